// Spatial half sweeps T(dts v_x d/dx) and T(dts v_y d/dy): exact splitting of A = v.grad_x into 1D
// advections, each a PFC flux-form remap, eqs. (38), (43)-(47) PAPER.md:247-295.
//
// Mapping: one thread owns VEC (=2) neighbouring v_z cells of ONE phase-space line and marches along
// the line with a 3-cell register window; a warp therefore reads/writes 512 contiguous bytes per line
// position.  The shift sigma = v_d dts / dx_d is uniform along a line, so the remap is "translate by
// n = floor|sigma| cells, then remap by the fraction b": out_i = f_j + (G_{j-u} - G_j), j = i - u n,
// u = sign(sigma), G = partial flux of eq. (46).  sigma < 0 (eq. 47 with the repaired sum, R5) is the
// same march on the mirrored line.  Out of place: src -> dst.
#include "vlasov_internal.cuh"

namespace vl {

struct SpaceParams {
    const double* __restrict__ src;
    double* __restrict__ dst;
    long S;            // doubles per spatial cell
    long line_stride;  // doubles between neighbours along the sweep (x: S, y: nx*S)
    int n_line;        // cells along the line that are UPDATED (x: nx, y: ny)
    int nx, ny, g, nyg;
    int nv1, nv2;      // nv[1], nv[2]
    int axis;          // 0: x sweep, 1: y sweep, 2: z sweep (3D3V, periodic)
    long slab;         // doubles per z slab (y sweep: blockIdx.z picks the slab)
    double vmin, dv;   // velocity direction that sets sigma
    double dts, dxx;
    double finf;
    int limiter;
    int bc_lo, bc_hi;
    int row0;          // x sweep: first ghost-inclusive row of this launch
    int* err;
};

template <int VEC> struct Pack;
template <> struct Pack<1> { double v[1]; };
template <> struct Pack<2> { double v[2]; };

template <int VEC>
__device__ __forceinline__ Pack<VEC> ld(const double* p) {
    Pack<VEC> r;
    if (VEC == 2) { double2 t = __ldcs(reinterpret_cast<const double2*>(p)); r.v[0] = t.x; r.v[VEC - 1] = t.y; }
    else r.v[0] = __ldcs(p);
    return r;
}
template <int VEC>
__device__ __forceinline__ void st(double* p, const Pack<VEC>& r) {
    if (VEC == 2) __stcs(reinterpret_cast<double2*>(p), make_double2(r.v[0], r.v[VEC - 1]));
    else __stcs(p, r.v[0]);
}

// Value(s) of line position r (any integer) of this thread's line.  base: pointer to position 0 of the
// line at this thread's velocity chunk; mir: offset (doubles) to the same cells with i_vy mirrored.
template <int VEC>
__device__ __forceinline__ Pack<VEC> fetch(const SpaceParams& P, const double* base, long mir, int r, bool& bad) {
    const int N = P.n_line;
    if (r >= 0 && r < N) return ld<VEC>(base + (long)r * P.line_stride);
    long off = 0;
    if (P.axis != 1) {                      // x, z: periodic
        while (r < 0) r += N;
        while (r >= N) r -= N;
        return ld<VEC>(base + (long)r * P.line_stride);
    }
    for (int guard = 0; guard < 4 && (r < 0 || r >= N); ++guard) {
        if (r < 0) {
            if (P.bc_lo == VLASOV_BC_PERIODIC) r += N;
            else if (P.bc_lo == VLASOV_BC_REFLECT) { r = -1 - r; off = (off == 0) ? mir : 0; }   // R19
            else { if (r + P.g < 0) { bad = true; Pack<VEC> z; z.v[0] = 0; z.v[VEC - 1] = 0; return z; }
                   return ld<VEC>(base + (long)r * P.line_stride + off); }                         // ghost row, R16
        } else {
            if (P.bc_hi == VLASOV_BC_PERIODIC) r -= N;
            else if (P.bc_hi == VLASOV_BC_REFLECT) { r = 2 * N - 1 - r; off = (off == 0) ? mir : 0; }
            else { if (r + P.g >= P.nyg) { bad = true; Pack<VEC> z; z.v[0] = 0; z.v[VEC - 1] = 0; return z; }
                   return ld<VEC>(base + (long)r * P.line_stride + off); }
        }
    }
    if (r < 0 || r >= N) { bad = true; Pack<VEC> z; z.v[0] = 0; z.v[VEC - 1] = 0; return z; }
    return ld<VEC>(base + (long)r * P.line_stride + off);
}

template <int VEC, int PF>
__global__ void __launch_bounds__(128) sweep_space_kernel(SpaceParams P) {
    const long chunks = P.S / VEC;
    const long chunk = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (chunk >= chunks) return;
    const long v = chunk * VEC;
    const int ivx = (int)(v / ((long)P.nv1 * P.nv2));
    const int ivy = (int)((v / P.nv2) % P.nv1);
    const int other = P.row0 + blockIdx.y;  // x sweep: row (of all slabs); y sweep: ix; z sweep: spatial cell of a slab
    const double* base;
    double* obase;
    long mir = 0;
    double vc;
    if (P.axis == 0) {
        base = P.src + ((long)other * P.nx) * P.S + v;
        obase = P.dst + ((long)other * P.nx) * P.S + v;
        vc = P.vmin + (ivx + 0.5) * P.dv;
    } else if (P.axis == 2) {
        base = P.src + (long)other * P.S + v;
        obase = P.dst + (long)other * P.S + v;
        vc = P.vmin + ((int)(v % P.nv2) + 0.5) * P.dv;      // the first v_z cell of this thread
    } else {
        const long zo = (long)blockIdx.z * P.slab;
        base = P.src + zo + ((long)P.g * P.nx + other) * P.S + v;
        obase = P.dst + zo + ((long)P.g * P.nx + other) * P.S + v;
        mir = (long)(P.nv1 - 1 - 2 * ivy) * P.nv2;
        vc = P.vmin + (ivy + 0.5) * P.dv;
        // ghost rows are Dirichlet data (R16): carried over unchanged
        for (int r = 0; r < P.g; ++r) {
            st<VEC>(P.dst + zo + ((long)r * P.nx + other) * P.S + v, ld<VEC>(P.src + zo + ((long)r * P.nx + other) * P.S + v));
            long rr = P.g + P.ny + r;
            st<VEC>(P.dst + zo + (rr * P.nx + other) * P.S + v, ld<VEC>(P.src + zo + (rr * P.nx + other) * P.S + v));
        }
    }
    const int N = P.n_line;
    const double sigma = vc * P.dts / P.dxx;
    int u = sigma >= 0.0 ? 1 : -1;
    int n; double b;
    split_shift(fabs(sigma), n, b);
    const bool periodic = P.axis != 1 || (P.bc_lo == VLASOV_BC_PERIODIC && P.bc_hi == VLASOV_BC_PERIODIC);
    if (periodic) n %= N;
    // shift fraction per packed cell: the same for both in x and y sweeps (sigma depends on i_vx / i_vy); in a z sweep
    // the two v_z cells of a thread have their own sigma -- the launcher packs two only when every |sigma_z| < 1 and
    // no pair straddles v_z = 0 (one direction, no whole cells)
    double bv[VEC];
#pragma unroll
    for (int e = 0; e < VEC; ++e) bv[e] = b;
    if (VEC == 2 && P.axis == 2) {
        const double s1 = (vc + P.dv) * P.dts / P.dxx;
        u = sigma + s1 >= 0.0 ? 1 : -1;
        n = 0;
        bv[0] = fabs(sigma); bv[VEC - 1] = fabs(s1);
    }
    bool bad = false;

    // march i = i0, i0+u, ...; source cell j = i - u n
    const int i0 = u > 0 ? 0 : N - 1;
    int j = i0 - u * n;
    Pack<VEC> fm = fetch<VEC>(P, base, mir, j - u, bad);
    Pack<VEC> f0 = fetch<VEC>(P, base, mir, j, bad);
    Pack<VEC> Gp;
    {
        Pack<VEC> fmm = fetch<VEC>(P, base, mir, j - 2 * u, bad);
#pragma unroll
        for (int e = 0; e < VEC; ++e) Gp.v[e] = partial_flux(fmm.v[e], fm.v[e], f0.v[e], bv[e], P.finf, P.limiter);
    }
    Pack<VEC> q[PF];
#pragma unroll
    for (int k = 0; k < PF; ++k) if (k < N) q[k] = fetch<VEC>(P, base, mir, j + u * (k + 1), bad);
    int i = i0;
    for (int t = 0; t < N; t += PF) {
#pragma unroll
        for (int k = 0; k < PF; ++k) {
            if (t + k < N) {
                Pack<VEC> fp = q[k];
                if (t + k + PF < N) q[k] = fetch<VEC>(P, base, mir, j + u * (PF + 1), bad);
                Pack<VEC> o;
#pragma unroll
                for (int e = 0; e < VEC; ++e) {
                    double G = partial_flux(fm.v[e], f0.v[e], fp.v[e], bv[e], P.finf, P.limiter);
                    o.v[e] = f0.v[e] + (Gp.v[e] - G);      // eq. (38): f + (Phi_{i-1/2} - Phi_{i+1/2})
                    Gp.v[e] = G;
                }
                st<VEC>(obase + (long)i * P.line_stride, o);
                fm = f0; f0 = fp;
                i += u; j += u;
            }
        }
    }
    if (bad) atomicCAS(P.err, 0, VLASOV_ESHIFT);
}

// z sweep of a short periodic line held in registers (3D3V, nz = NZ, every |sigma_z| < 1 and no pair of v_z cells
// straddling v_z = 0): a thread owns two neighbouring v_z cells of one spatial column (ix, iy) and all NZ slabs of them.
// All 2 NZ values are loaded at once (NZ independent 16-byte loads in flight), in the direction of the flow -- eq. (47)
// is eq. (46) on the mirrored line -- so position i of the window is slab i (sigma >= 0) or NZ-1-i (sigma < 0); the
// wrap-around is a compile-time index.  The general kernel above spends a short line on its prefetch queue and the
// run-time wrap (0.50 of the HBM peak on 8 slabs).
template <int NZ>
__global__ void __launch_bounds__(128) sweep_z_reg_kernel(SpaceParams P) {
    const long chunk = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (chunk >= P.S / 2) return;
    const long v = chunk * 2;
    const long col = (long)blockIdx.y * P.S + v;
    const double va = P.vmin + ((int)(v % P.nv2) + 0.5) * P.dv;
    const double sa = va * P.dts / P.dxx, sb = (va + P.dv) * P.dts / P.dxx;
    const bool pos = sa + sb >= 0.0;
    const double ba = fabs(sa), bb = fabs(sb);
    double qa[NZ], qb[NZ];
#pragma unroll
    for (int i = 0; i < NZ; ++i) {
        const double2 t = __ldcs(reinterpret_cast<const double2*>(P.src + col + (long)(pos ? i : NZ - 1 - i) * P.slab));
        qa[i] = t.x; qb[i] = t.y;
    }
    double Ga[NZ], Gb[NZ];          // flux out of position i (through its downstream face)
#pragma unroll
    for (int i = 0; i < NZ; ++i) {
        const int im = (i + NZ - 1) % NZ, ip = (i + 1) % NZ;
        Ga[i] = partial_flux(qa[im], qa[i], qa[ip], ba, P.finf, P.limiter);
        Gb[i] = partial_flux(qb[im], qb[i], qb[ip], bb, P.finf, P.limiter);
    }
#pragma unroll
    for (int i = 0; i < NZ; ++i) {
        const int im = (i + NZ - 1) % NZ;
        const double2 o = make_double2(qa[i] + (Ga[im] - Ga[i]), qb[i] + (Gb[im] - Gb[i]));      // eq. (38)
        __stcs(reinterpret_cast<double2*>(P.dst + col + (long)(pos ? i : NZ - 1 - i) * P.slab), o);
    }
}

static int launch_space(vlasov_ctx* c, const Species& s, const double* src, double* dst, double dts, int axis,
                        int row0 = 0, int nrows = -1) {
    const Geom& G = c->G;
    SpaceParams P;
    P.src = src; P.dst = dst;
    P.S = s.nvtot;
    P.axis = axis;
    P.nx = G.nx; P.ny = G.ny; P.g = G.g; P.nyg = G.nyg;
    P.nv1 = s.nv[1]; P.nv2 = s.nv[2];
    P.slab = (long)G.nyg * G.nx * s.nvtot;
    P.line_stride = axis == 0 ? s.nvtot : axis == 1 ? (long)G.nx * s.nvtot : P.slab;
    P.n_line = axis == 0 ? G.nx : axis == 1 ? G.ny : G.nz;
    P.vmin = s.vmin[axis]; P.dv = s.dv[axis];
    P.dts = dts; P.dxx = axis == 0 ? G.dx : axis == 1 ? G.dy : G.dz;
    P.finf = s.f_inf; P.limiter = G.limiter;
    P.bc_lo = G.bc_lo; P.bc_hi = G.bc_hi;
    P.err = c->errflag;
    P.row0 = axis == 0 ? row0 : 0;
    if (nrows < 0) nrows = G.nrows;              // x sweep: the rows of every z slab
    if (nrows == 0) return VLASOV_OK;
    const int threads = 128;
    if (axis == 2) {                             // sigma depends on i_vz
        // two v_z cells per thread (16-byte accesses) when both march the same way with no whole cells, else one
        bool pack = s.nv[2] % 2 == 0;
        for (int k = 0; k + 1 < s.nv[2] && pack; k += 2) {
            const double s0 = (s.vmin[2] + (k + 0.5) * s.dv[2]) * dts / G.dz, s1 = (s.vmin[2] + (k + 1.5) * s.dv[2]) * dts / G.dz;
            pack = s0 * s1 >= 0.0 && fabs(s0) < 1.0 && fabs(s1) < 1.0;
        }
        Launch L(c, K_SWEEP_Z);
        if (pack) {
            dim3 grid((unsigned)((s.nvtot / 2 + threads - 1) / threads), (unsigned)(G.nyg * G.nx));
            if (G.nz == 8) sweep_z_reg_kernel<8><<<grid, threads, 0, c->stream>>>(P);
            else if (G.nz == 4) sweep_z_reg_kernel<4><<<grid, threads, 0, c->stream>>>(P);
            else if (G.nz == 16) sweep_z_reg_kernel<16><<<grid, threads, 0, c->stream>>>(P);
            else sweep_space_kernel<2, 4><<<grid, threads, 0, c->stream>>>(P);
        } else {
            dim3 grid((unsigned)((s.nvtot + threads - 1) / threads), (unsigned)(G.nyg * G.nx));
            sweep_space_kernel<1, 4><<<grid, threads, 0, c->stream>>>(P);
        }
    } else {
        // two neighbouring v_z cells per thread (one sigma, one wall image, 16-byte accesses) need an even nv[2]
        const bool pack = s.nv[2] % 2 == 0;
        const long chunks = pack ? s.nvtot / 2 : s.nvtot;
        dim3 grid((unsigned)((chunks + threads - 1) / threads), (unsigned)(axis == 0 ? nrows : G.nx), (unsigned)(axis == 0 ? 1 : G.nz));
        Launch L(c, axis == 0 ? K_SWEEP_X : K_SWEEP_Y);
        if (pack) sweep_space_kernel<2, 4><<<grid, threads, 0, c->stream>>>(P);
        else sweep_space_kernel<1, 4><<<grid, threads, 0, c->stream>>>(P);
    }
    return cudaGetLastError() == cudaSuccess ? VLASOV_OK : VLASOV_ECUDA;
}

int launch_sweep_x(vlasov_ctx* c, const Species& s, const double* src, double* dst, double dts) {
    return launch_space(c, s, src, dst, dts, 0);
}
int launch_sweep_x_rows(vlasov_ctx* c, const Species& s, const double* src, double* dst, double dts, int row0, int nrows) {
    return launch_space(c, s, src, dst, dts, 0, row0, nrows);
}
int launch_sweep_y(vlasov_ctx* c, const Species& s, const double* src, double* dst, double dts) {
    return launch_space(c, s, src, dst, dts, 1);
}
int launch_sweep_z(vlasov_ctx* c, const Species& s, const double* src, double* dst, double dts) {
    return launch_space(c, s, src, dst, dts, 2);
}

}  // namespace vl
