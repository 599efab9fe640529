// a9: velocity moments, eqs. (2)-(4) PAPER.md:39-46 as midpoint sums over the velocity block of one
// spatial cell (R14: the 10 raw moments M0, M1_d, M2_de, each times dvx dvy dvz), plus max_v f as an
// 11th output (the ghost fill's f_infinity, R15d).  Current density, eq. (11) PAPER.md:74.
//
// One CTA per spatial cell.  A thread owns pairs of neighbouring v_z cells and walks i_vx with three
// running sums per column (sum f, sum vx f, sum vx^2 f), folded with (vy, vz) once per column: about
// 3.3 fp64 operations per phase-space cell.  Reduction: warp shuffle, then a fixed-order tree over the
// warps in shared memory -- no atomics, so reruns are bit-identical.
#include "vlasov_internal.cuh"

namespace vl {

struct MomParams {
    const double* __restrict__ f;
    double* __restrict__ out;   // [11][ncell_out]
    long S;
    int nv0, nv1, nv2;
    double vmin[3], dv[3];
    int cell0, ncell_out;
};

constexpr int MOM_THREADS = 256;

// VEC = 2: a thread owns pairs of neighbouring v_z cells (16-byte loads; nv[2] even).  VEC = 1: one column per thread
// (any nv[2]); the same sums in the same order per column.
template <int VEC, int NT = MOM_THREADS>
__global__ void __launch_bounds__(NT) moments_kernel(MomParams P) {
    const int cell = P.cell0 + blockIdx.x;
    const double* fb = P.f + (long)cell * P.S;
    const int plane = P.nv1 * P.nv2;
    const int nchunk = plane / VEC;
    double M[10];
#pragma unroll
    for (int k = 0; k < 10; ++k) M[k] = 0.0;
    double mx = 0.0;
    for (int ch = threadIdx.x; ch < nchunk; ch += NT) {
        const int col = VEC * ch;
        const int iy = col / P.nv2, iz = col - iy * P.nv2;
        const double vy = P.vmin[1] + (iy + 0.5) * P.dv[1];
        const double vza = P.vmin[2] + (iz + 0.5) * P.dv[2];
        const double vzb = P.vmin[2] + (iz + 1.5) * P.dv[2];
        double a0 = 0, a1 = 0, a2 = 0, b0 = 0, b1 = 0, b2 = 0;
        if constexpr (VEC == 2) {
            const double2* p = reinterpret_cast<const double2*>(fb + col);
            const long pstride = plane / 2;
#pragma unroll 4
            for (int k = 0; k < P.nv0; ++k) {
                const double vx = P.vmin[0] + (k + 0.5) * P.dv[0];
                const double2 v = __ldcs(p + (long)k * pstride);
                const double wa = vx * v.x, wb = vx * v.y;
                a0 += v.x; a1 += wa; a2 += vx * wa;
                b0 += v.y; b1 += wb; b2 += vx * wb;
                mx = fmax(mx, fmax(v.x, v.y));
            }
        } else {
            const double* p = fb + col;
#pragma unroll 4
            for (int k = 0; k < P.nv0; ++k) {
                const double vx = P.vmin[0] + (k + 0.5) * P.dv[0];
                const double v = __ldcs(p + (long)k * plane);
                const double wa = vx * v;
                a0 += v; a1 += wa; a2 += vx * wa;
                mx = fmax(mx, v);
            }
        }
        const double s0 = a0 + b0, s1 = a1 + b1, s2 = a2 + b2;
        const double z0 = vza * a0 + vzb * b0;          // sum vz f
        const double z1 = vza * a1 + vzb * b1;          // sum vx vz f
        M[0] += s0;
        M[1] += s1;
        M[2] += vy * s0;
        M[3] += z0;
        M[4] += s2;
        M[5] += vy * vy * s0;
        M[6] += vza * vza * a0 + vzb * vzb * b0;
        M[7] += vy * s1;
        M[8] += z1;
        M[9] += vy * z0;
    }
    // warp tree
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
#pragma unroll
        for (int k = 0; k < 10; ++k) M[k] += __shfl_down_sync(0xffffffffu, M[k], o);
        mx = fmax(mx, __shfl_down_sync(0xffffffffu, mx, o));
    }
    __shared__ double red[MOM_THREADS / 32][11];
    const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
    if (l == 0) {
#pragma unroll
        for (int k = 0; k < 10; ++k) red[w][k] = M[k];
        red[w][10] = mx;
    }
    __syncthreads();
    if (threadIdx.x < 11) {
        const int k = threadIdx.x;
        double r = red[0][k];
        for (int ww = 1; ww < NT / 32; ++ww) r = (k < 10) ? r + red[ww][k] : fmax(r, red[ww][k]);
        if (k < 10) r *= P.dv[0] * P.dv[1] * P.dv[2];
        P.out[(long)k * P.ncell_out + blockIdx.x] = r;
    }
}

int launch_moments(vlasov_ctx* c, const Species& s, const double* f, double* out, int row0, int nrows) {
    if (nrows <= 0) return VLASOV_OK;
    MomParams P;
    P.f = f; P.out = out; P.S = s.nvtot;
    P.nv0 = s.nv[0]; P.nv1 = s.nv[1]; P.nv2 = s.nv[2];
    for (int d = 0; d < 3; ++d) { P.vmin[d] = s.vmin[d]; P.dv[d] = s.dv[d]; }
    P.cell0 = row0 * c->G.nx;
    P.ncell_out = nrows * c->G.nx;
    {
        Launch L(c, K_MOMENTS);
        // Small velocity planes (fewer than two trips of MOM_THREADS threads: 16^3 has 128 pairs of columns, 24^3 288)
        // get a CTA whose threads the columns divide evenly among -- measured 0.091 -> 0.074 ms (16^3) and 0.223 -> 0.202 ms
        // (24^3) per cycle of config 5.  Larger planes keep MOM_THREADS: other resident CTAs fill a ragged last trip, and
        // smaller CTAs measured slower there (40^3: 1.67 -> 2.03 ms).
        const int nchunk = s.nv[1] * s.nv[2] / (s.nv[2] % 2 == 0 ? 2 : 1);
        auto waste = [&](int t) { return ((nchunk + t - 1) / t) * t - nchunk; };
        int nt = MOM_THREADS;
        if (waste(192) == 0 && waste(nt) > 0) nt = 192;      // 48^3: 1152 pairs of columns = 6 x 192 (1.19 -> 1.12 ms)
        if (nchunk < 2 * MOM_THREADS) {
            if (waste(128) < waste(nt)) nt = 128;
            if (waste(96) < waste(nt)) nt = 96;
        }
        if (s.nv[2] % 2 == 0) {
            if (nt == 192) moments_kernel<2, 192><<<P.ncell_out, 192, 0, c->stream>>>(P);
            else if (nt == 128) moments_kernel<2, 128><<<P.ncell_out, 128, 0, c->stream>>>(P);
            else if (nt == 96) moments_kernel<2, 96><<<P.ncell_out, 96, 0, c->stream>>>(P);
            else moments_kernel<2><<<P.ncell_out, MOM_THREADS, 0, c->stream>>>(P);
        } else {
            moments_kernel<1><<<P.ncell_out, MOM_THREADS, 0, c->stream>>>(P);
        }
    }
    return cudaGetLastError() == cudaSuccess ? VLASOV_OK : VLASOV_ECUDA;
}

// max over an array (one block; fmax is exact, so the order does not matter): f_infinity := max f at init (R6)
__global__ void __launch_bounds__(256) max_kernel(const double* __restrict__ a, long n, double* __restrict__ out) {
    __shared__ double red[256];
    double m = a[0];
    for (long i = threadIdx.x; i < n; i += 256) m = fmax(m, a[i]);
    red[threadIdx.x] = m;
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o) red[threadIdx.x] = fmax(red[threadIdx.x], red[threadIdx.x + o]);
        __syncthreads();
    }
    if (threadIdx.x == 0) *out = red[0];
}

// max of f over every cell of one species, through the 11th output of the moments kernel; synchronises the stream
int species_max_f(vlasov_ctx* c, const Species& s, double* result) {
    const int ncell = c->G.nrows * c->G.nx;
    int e = launch_moments(c, s, s.f, c->mom, 0, c->G.nrows);
    if (e) return e;
    max_kernel<<<1, 256, 0, c->stream>>>(c->mom + (long)10 * ncell, ncell, c->gmom);
    if (cudaMemcpyAsync(result, c->gmom, sizeof(double), cudaMemcpyDeviceToHost, c->stream) != cudaSuccess) return VLASOV_ECUDA;
    if (cudaStreamSynchronize(c->stream) != cudaSuccess) return VLASOV_ECUDA;
    return VLASOV_OK;
}

// ------------------------------------------------------------------------------------------------
// Section 4.1: "by linear interpolation in time": out = (1 - theta) a + theta b, two products and a
// sum, each rounded (no contraction), as the oracle writes it.
// ------------------------------------------------------------------------------------------------
__global__ void lerp_kernel(const double* __restrict__ a, const double* __restrict__ b, double theta, double* __restrict__ out, long n) {
    const long i = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) out[i] = __dadd_rn(__dmul_rn(1.0 - theta, a[i]), __dmul_rn(theta, b[i]));
}

int launch_lerp(vlasov_ctx* c, const double* a, const double* b, double theta, double* out, long n) {
    if (n <= 0) return VLASOV_OK;
    {
        Launch L(c, K_MOMENTS);
        lerp_kernel<<<(unsigned)((n + 255) / 256), 256, 0, c->stream>>>(a, b, theta, out, n);
    }
    return cudaGetLastError() == cudaSuccess ? VLASOV_OK : VLASOV_ECUDA;
}

// rows [off, off + n) of each of nk moment planes of src [nk][src_stride] -> dst [nk][n] (the border rows of the kept
// moments: section 4.1 needs no second pass over f when the step has just reduced them)
__global__ void gather_rows_kernel(const double* __restrict__ src, long src_stride, long off, double* __restrict__ dst, long n, int nk) {
    const long i = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n * nk) return;
    const long k = i / n, j = i - k * n;
    dst[i] = src[k * src_stride + off + j];
}

int launch_gather_rows(vlasov_ctx* c, const double* src, long src_stride, long off, double* dst, long n, int nk) {
    if (n <= 0) return VLASOV_OK;
    {
        Launch L(c, K_MOMENTS);
        gather_rows_kernel<<<(unsigned)((n * nk + 255) / 256), 256, 0, c->stream>>>(src, src_stride, off, dst, n, nk);
    }
    return cudaGetLastError() == cudaSuccess ? VLASOV_OK : VLASOV_ECUDA;
}

// ------------------------------------------------------------------------------------------------
// eq. (11): j = sum_s q_s M1^(s); Yee: interpolated to the E positions of R17
// ------------------------------------------------------------------------------------------------
struct CurParams {
    const double* __restrict__ mom;   // [ns][11][ncell]
    double* __restrict__ J;
    double q[MAX_SPECIES];
    int ns, nx, nyg, nz, fields_yee, wall;
};

__device__ __forceinline__ double jc_at(const CurParams& P, int d, int k, int j, int i) {
    const long PL = (long)P.nx * P.nyg * P.nz;
    double r = 0.0;
    for (int s = 0; s < P.ns; ++s) r += P.q[s] * P.mom[((long)s * 11 + 1 + d) * PL + ((long)k * P.nyg + j) * P.nx + i];
    return r;
}

// J at the E positions of the Yee grid (R17 / R24): Jx(i+1/2,j,k) averages the cell-centre currents over (j-1,j) x
// (k-1,k), Jy(i,j+1/2,k) over (i-1,i) x (k-1,k), Jz(i,j,k+1/2) over (i-1,i) x (j-1,j).  With nz = 1 the z neighbour
// is the cell itself and the sums are the 2D ones bit for bit.
__global__ void current_kernel(CurParams P) {
    const int cell = blockIdx.x * blockDim.x + threadIdx.x;
    const int ncell = P.nx * P.nyg * P.nz;
    if (cell >= ncell) return;
    const int i = cell % P.nx, j = (cell / P.nx) % P.nyg, k = cell / (P.nx * P.nyg);
    const long PL = ncell;
    if (!P.fields_yee) {
        for (int d = 0; d < 3; ++d) P.J[d * PL + cell] = jc_at(P, d, k, j, i);
        return;
    }
    const int im = (i + P.nx - 1) % P.nx, km = (k + P.nz - 1) % P.nz;
    int jm = j - 1;
    bool onwall = false;
    if (jm < 0) { jm = P.nyg - 1; onwall = P.wall != 0; }
    P.J[0 * PL + cell] = onwall ? 0.0 : 0.25 * ((jc_at(P, 0, km, jm, i) + jc_at(P, 0, km, j, i)) + (jc_at(P, 0, k, jm, i) + jc_at(P, 0, k, j, i)));
    P.J[1 * PL + cell] = 0.25 * ((jc_at(P, 1, km, j, im) + jc_at(P, 1, km, j, i)) + (jc_at(P, 1, k, j, im) + jc_at(P, 1, k, j, i)));
    P.J[2 * PL + cell] = onwall ? 0.0 : 0.25 * (jc_at(P, 2, k, jm, im) + jc_at(P, 2, k, jm, i) + jc_at(P, 2, k, j, im) + jc_at(P, 2, k, j, i));
}

int launch_current(vlasov_ctx* c, double* J) {
    CurParams P;
    P.mom = c->mom; P.J = J;
    P.ns = c->ns; P.nx = c->G.nx; P.nyg = c->G.nyg; P.nz = c->G.nz; P.fields_yee = c->G.fields_yee; P.wall = c->G.wall;
    for (int s = 0; s < c->ns; ++s) P.q[s] = c->sp[s].q;
    const int ncell = P.nx * P.nyg * P.nz;
    {
        Launch L(c, K_CURRENT);
        current_kernel<<<(ncell + 127) / 128, 128, 0, c->stream>>>(P);
    }
    return cudaGetLastError() == cudaSuccess ? VLASOV_OK : VLASOV_ECUDA;
}

}  // namespace vl
