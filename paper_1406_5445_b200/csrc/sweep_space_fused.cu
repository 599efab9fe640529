// Fused spatial half steps: T(dts v_x d/dx) T(dts v_y d/dy) in ONE pass over f (a1+a2), and the palindromic
// T(dts v_y d/dy) T(dts v_x d/dx) (a7+a8) -- the exact splitting of A = v.grad_x into 1D advections
// (PAPER.md:156), each a PFC flux-form remap, eqs. (38), (43)-(47) PAPER.md:247-295.  Used when every
// shift of the stage is below one cell (|sigma| < 1: the whole-cell sums of eqs. (46)/(47) are empty);
// otherwise api.cu falls back to the general one-direction kernels of sweep_space.cu.
//
// Mapping.  A CTA owns C contiguous velocity cells of every
// spatial cell and marches over the rows (y) of the block:
//   * a thread owns XB consecutive x cells of one velocity cell; its warp reads/writes C*8 contiguous
//     bytes per (x, y);
//   * x couples threads: the row's values go through a double-buffered shared row [x][c] and each thread
//     reads the 3 halo cells of its x block (periodic wrap);
//   * y is private to a thread: a 2-cell register window plus the previous flux per owned cell.
// Rows -2, -1 and ny, ny+1 are the boundary rows of the y sweep (R16, R19): periodic wrap, the wall
// image f(y_w + eta, vy) = f(y_w - eta, -vy), or FLUID ghost rows; they are loaded like any row.
#include "vlasov_internal.cuh"

namespace vl {

struct XYParams {
    const double* __restrict__ src;
    double* __restrict__ dst;
    long S;            // doubles per spatial cell
    long row_stride;   // nx * S
    int nx, ny, g;
    int nv1, nv2;
    int C;             // contiguous velocity cells per CTA
    int PC;            // cells per bulk copy (a piece of one v_z row, or the whole chunk)
    double vminx, dvx, vminy, dvy;
    double kx, ky;     // dts/dx, dts/dy
    double finf;
    int bc_lo, bc_hi;
};

// ---- 1D bulk TMA (cp.async.bulk) + mbarrier: rows land in shared memory without passing registers ----
__device__ __forceinline__ void mbar_init(unsigned bar, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(unsigned bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned bar, unsigned parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_LOOP:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE;\n"
        "bra WAIT_LOOP;\n"
        "DONE:\n"
        "}\n" ::"r"(bar), "r"(parity) : "memory");
}
__device__ __forceinline__ void bulk_g2s(unsigned dst, const void* src, unsigned bytes, unsigned bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}

struct Weights {
    double w0, w1, w2;     // alpha, alpha (1-a)(2-a)/6, alpha (1-a)(1+a)/6 of eq. (46): uniform along a line
    bool pos;
    __device__ __forceinline__ void set(double sigma) {
        pos = sigma >= 0.0;
        const double b = fabs(sigma);
        w0 = b;
        w1 = b * ((1.0 - b) * (2.0 - b) * (1.0 / 6.0));
        w2 = b * ((1.0 - b) * (1.0 + b) * (1.0 / 6.0));
    }
};

// Does the slope pair (dp, dm) of a cell with value f0 possibly need limiting?  High-word test of
// vlasov_internal.cuh (conservative).  Returns a word whose sign bit is set if so.
__device__ __forceinline__ int need_bits(double f0, double dp, double dm, double finf) {
    const int hb = min(__double2hiint(f0), __double2hiint(finf - f0)) + 0x00100000;
    const int hp = __double2hiint(dp) & 0x7fffffff, hm = __double2hiint(dm) & 0x7fffffff;
    return (hb - 1) - max(hp, hm);
}

// N partial fluxes alpha [ f0 + c1 eps+ d+ + c2 eps- d- ] of the cells q[1..N] of a line piece q[0..N+1]
// (q ordered in the direction of the flow, so eq. (47) is the same call on the reversed piece).
// The limiter test is batched: one vote per call, and the usual answer is "nobody".
template <int N, int LIM>
__device__ __forceinline__ void flux_line(const double (&q)[N + 2], const Weights& W, double finf, double (&G)[N]) {
    double d[N + 1];
#pragma unroll
    for (int i = 0; i <= N; ++i) d[i] = q[i + 1] - q[i];
    if (LIM) {
        int need = 0;
#pragma unroll
        for (int i = 0; i < N; ++i) need |= need_bits(q[i + 1], d[i + 1], d[i], finf);
        if (__any_sync(__activemask(), need < 0)) {
#pragma unroll
            for (int i = 0; i < N; ++i) {
                double sp, sm;
                slopes_fast<1>(q[i], q[i + 1], q[i + 2], finf, sp, sm);
                G[i] = fma(W.w2, sm, fma(W.w1, sp, W.w0 * q[i + 1]));
            }
            return;
        }
    }
#pragma unroll
    for (int i = 0; i < N; ++i) G[i] = fma(W.w2, d[i], fma(W.w1, d[i + 1], W.w0 * q[i + 1]));
}

// x remap of CH of the XB owned cells of one row (chunk k along the flow); the row sits in shared memory at
// sbuf ([x][c], this thread's column at byte offset cofs).  DIR = +1: sigma >= 0, eq. (46); DIR = -1: eq. (47),
// the same on the mirrored line.  val[i] = new average, eq. (38), of owned cell item(k, i); the flux through
// the chunk border is carried over (same arithmetic on the same inputs: identical value).
template <int XB, int CH, int DIR>
__device__ __forceinline__ int x_item(int k, int i) { return DIR > 0 ? k * CH + i : XB - 1 - (k * CH + i); }

template <int XB, int CH, int LIM, int DIR>
__device__ __forceinline__ void x_chunk(int k, double& carry, double (&val)[CH], unsigned sbuf, int ix0, int nx, int C8,
                                        unsigned cofs, const Weights& W, double finf) {
    // position p = 0 .. XB+2 along the flow: cell ix0-2+p (DIR > 0) or ix0+XB+1-p (DIR < 0)
    double q[CH + 3], G[CH + 1];
#pragma unroll
    for (int i = 0; i < CH + 3; ++i) {
        const int p = k * CH + i;
        int ix = DIR > 0 ? ix0 - 2 + p : ix0 + XB + 1 - p;
        if (p < 2 || p == XB + 2) { if (ix < 0) ix += nx; else if (ix >= nx) ix -= nx; }
        q[i] = lds(sbuf + ix * C8 + cofs);
    }
    flux_line<CH + 1, LIM>(q, W, finf, G);         // fluxes out of positions 1+k CH .. 1+k CH+CH
    if (k > 0) G[0] = carry;
    carry = G[CH];
#pragma unroll
    for (int i = 0; i < CH; ++i) val[i] = q[i + 2] + (G[i] - G[i + 1]);
}

// One step of the y march of an owned cell: rows (r-2, r-1, r) = (ya, yb, gx) -> new average h of row r-1
// (sigma_y >= 0, eq. 46) or r-2 (sigma_y < 0, eq. 47 on the mirrored line).
template <int LIM>
__device__ __forceinline__ double y_step(double& ya, double& yb, double& yG, double gx, const Weights& Wy, double finf) {
    const double dlo = yb - ya, dhi = gx - yb;
    double sp = Wy.pos ? dhi : -dlo, sm = Wy.pos ? dlo : -dhi;
    if (LIM) {
        if (__any_sync(__activemask(), need_bits(yb, dhi, dlo, finf) < 0)) {
            if (Wy.pos) slopes_fast<1>(ya, yb, gx, finf, sp, sm); else slopes_fast<1>(gx, yb, ya, finf, sp, sm);
        }
    }
    const double Gn = fma(Wy.w2, sm, fma(Wy.w1, sp, Wy.w0 * yb));
    const double h = Wy.pos ? yb + (yG - Gn) : ya + (Gn - yG);
    yG = Gn; ya = yb; yb = gx;
    return h;
}

// Array row and image flag of boundary-inclusive row r (-2 <= r <= ny+1) of the y sweep.
__device__ __forceinline__ int virtual_row(const XYParams& P, int r, bool& mirror) {
    mirror = false;
    if (r < 0) {
        if (P.bc_lo == VLASOV_BC_PERIODIC) r += P.ny;
        else if (P.bc_lo == VLASOV_BC_REFLECT) { r = -1 - r; mirror = true; }
    } else if (r >= P.ny) {
        if (P.bc_hi == VLASOV_BC_PERIODIC) r -= P.ny;
        else if (P.bc_hi == VLASOV_BC_REFLECT) { r = 2 * P.ny - 1 - r; mirror = true; }
    }
    return P.g + r;       // FLUID: the ghost row itself (R16)
}

// XFIRST = 1: x remap of every incoming row, then the y march (a1 + a2).
// XFIRST = 0: y march on the raw rows, then the x remap of every finished row (a7 + a8).
// Shared memory: [2 mbarriers][raw row 0][raw row 1]([y-swept row 0][y-swept row 1] if !XFIRST).
template <int XB, int LIM, int XFIRST>
__global__ void __launch_bounds__(512, 1) sweep_xy_kernel(XYParams P) {
    extern __shared__ __align__(128) unsigned char smraw[];
    const int C = P.C, C8 = C * 8;
    const int c = threadIdx.x % C, blk = threadIdx.x / C;
    const int ix0 = blk * XB;
    const long v0 = (long)blockIdx.x * C;
    const long v = v0 + c;
    const int ivx = (int)(v / ((long)P.nv1 * P.nv2));
    const int ivy = (int)((v / P.nv2) % P.nv1);
    Weights Wx, Wy;
    Wx.set((P.vminx + (ivx + 0.5) * P.dvx) * P.kx);
    Wy.set((P.vminy + (ivy + 0.5) * P.dvy) * P.ky);
    const unsigned bar0 = smem_addr(smraw);
    const unsigned rowbytes = (unsigned)P.nx * C8;
    const unsigned raw0 = bar0 + 128;
    const unsigned hb0 = raw0 + 2 * rowbytes;
    const unsigned cofs = c * 8;
    const unsigned own = (unsigned)ix0 * C8 + cofs;
    const double finf = P.finf;

    // producer side: piece t of a row = PC contiguous cells of one x (a v_z row or a part of one, so that its
    // wall image is contiguous too); the pieces are spread over the threads
    const int PC = P.PC, npp = C / PC;               // pieces per x
    const int ncopy = P.nx * npp;
    auto issue_row = [&](int r) {
        const unsigned bar = bar0 + 8 * (r & 1);
        if (threadIdx.x == 0) mbar_expect_tx(bar, rowbytes);
        bool m; const int ar = virtual_row(P, r, m);
        for (int t = threadIdx.x; t < ncopy; t += blockDim.x) {
            const int cp_ix = t / npp, cp_pc = t - cp_ix * npp;
            const long vp = v0 + (long)cp_pc * PC;
            long src = (long)ar * P.row_stride + (long)cp_ix * P.S + vp;
            if (m) src += (long)(P.nv1 - 1 - 2 * (int)((vp / P.nv2) % P.nv1)) * P.nv2;     // i_vy mirrored (R19)
            bulk_g2s(raw0 + (r & 1) * rowbytes + (unsigned)(cp_ix * C + cp_pc * PC) * 8, P.src + src, (unsigned)PC * 8, bar);
        }
    };
    if (threadIdx.x == 0) { mbar_init(bar0, 1); mbar_init(bar0 + 8, 1); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    __syncthreads();
    // thread 0 arms the barrier before any copy of that row can complete: the arming and the copies of a
    // row are issued after the same __syncthreads, thread 0's expect_tx first within its warp
    issue_row(-2);
    issue_row(-1);

    double ya[XB], yb[XB], yG[XB];
#pragma unroll
    for (int i = 0; i < XB; ++i) { ya[i] = 0.0; yb[i] = 0.0; yG[i] = 0.0; }
    const int orow_shift = Wy.pos ? 1 : 2;
    for (int r = -2; r <= P.ny + 1; ++r) {
        const int st = r & 1;
        const unsigned sraw = raw0 + st * rowbytes;
        mbar_wait(bar0 + 8 * st, ((r + 2) >> 1) & 1);
        const int orow = r - orow_shift;
        double* po = P.dst + (long)(P.g + orow) * P.row_stride + (long)ix0 * P.S + v;
        const bool store = orow >= 0 && orow < P.ny;
        constexpr int CH = XB < 4 ? XB : 4;
        if (XFIRST) {
            double carry = 0.0;
#pragma unroll
            for (int k = 0; k < XB / CH; ++k) {
                double gx[CH];
                if (Wx.pos) x_chunk<XB, CH, LIM, 1>(k, carry, gx, sraw, ix0, P.nx, C8, cofs, Wx, finf);
                else        x_chunk<XB, CH, LIM, -1>(k, carry, gx, sraw, ix0, P.nx, C8, cofs, Wx, finf);
#pragma unroll
                for (int i = 0; i < CH; ++i) {
                    // the item index is a compile-time constant on either branch
                    if (Wx.pos) {
                        constexpr int dummy = 0; (void)dummy;
                        const int it = k * CH + i;
                        const double h = y_step<LIM>(ya[it], yb[it], yG[it], gx[i], Wy, finf);
                        if (store) __stcs(po + (long)it * P.S, h);
                    } else {
                        const int it = XB - 1 - (k * CH + i);
                        const double h = y_step<LIM>(ya[it], yb[it], yG[it], gx[i], Wy, finf);
                        if (store) __stcs(po + (long)it * P.S, h);
                    }
                }
            }
            __syncthreads();                       // everybody is done reading raw row r
            if (r + 2 <= P.ny + 1) issue_row(r + 2);
        } else {
            const unsigned sh = hb0 + st * rowbytes;
#pragma unroll
            for (int i = 0; i < XB; ++i) {
                const double h = y_step<LIM>(ya[i], yb[i], yG[i], lds(sraw + own + i * C8), Wy, finf);
                sts(sh + own + i * C8, h);
            }
            __syncthreads();                       // y-swept row complete; raw row r free
            if (r + 2 <= P.ny + 1) issue_row(r + 2);
            double carry = 0.0;
#pragma unroll
            for (int k = 0; k < XB / CH; ++k) {
                double o[CH];
                if (Wx.pos) x_chunk<XB, CH, LIM, 1>(k, carry, o, sh, ix0, P.nx, C8, cofs, Wx, finf);
                else        x_chunk<XB, CH, LIM, -1>(k, carry, o, sh, ix0, P.nx, C8, cofs, Wx, finf);
                if (store) {
#pragma unroll
                    for (int i = 0; i < CH; ++i) {
                        const int it = Wx.pos ? k * CH + i : XB - 1 - (k * CH + i);
                        __stcs(po + (long)it * P.S, o[i]);
                    }
                }
            }
        }
    }
}

template <int XB, int LIM>
static void launch_xy_t(const XYParams& P, int xfirst, dim3 grid, int threads, size_t smem, cudaStream_t st) {
    if (xfirst) {
        cudaFuncSetAttribute(sweep_xy_kernel<XB, LIM, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        sweep_xy_kernel<XB, LIM, 1><<<grid, threads, smem, st>>>(P);
    } else {
        cudaFuncSetAttribute(sweep_xy_kernel<XB, LIM, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        sweep_xy_kernel<XB, LIM, 0><<<grid, threads, smem, st>>>(P);
    }
}

// Tile shape of the fused stage: XB x cells per thread, C contiguous velocity cells per CTA -- a power of two
// that divides the block, made of whole v_z rows or a part of one, at least 16 bytes, at most 512 threads.
static bool pick_xy_shape(const Geom& G, const Species& s, int& xb, int& C) {
    xb = 1;
    if (G.nx % 8 == 0) xb = 8; else if (G.nx % 4 == 0) xb = 4;
    const int nblk = G.nx / xb;
    C = 32;
    auto ok = [&](int cc) { return s.nvtot % cc == 0 && (s.nv[2] % cc == 0 || cc % s.nv[2] == 0) && nblk * cc <= 512; };
    while (C >= 2 && !ok(C)) C >>= 1;
    if (C < 2) return false;
    return 128 + 4 * (size_t)G.nx * C * 8 <= 200 * 1024;
}

// Whether the fused stage applies: all shifts below one cell, at least two cells per direction, two ghost
// rows where a side is FLUID (otherwise the general kernels run and report ESHIFT where due), a tile shape.
bool fused_xy_applicable(const vlasov_ctx* c, const Species& s, double dts) {
    const Geom& G = c->G;
    if (G.nx < 2 || G.ny < 2) return false;
    if ((G.bc_lo == VLASOV_BC_FLUID || G.bc_hi == VLASOV_BC_FLUID) && G.g < 2) return false;
    for (int d = 0; d < 2; ++d) {
        const double vlo = fabs(s.vmin[d] + 0.5 * s.dv[d]);
        const double vhi = fabs(s.vmin[d] + (s.nv[d] - 0.5) * s.dv[d]);
        const double vmax = vlo > vhi ? vlo : vhi;
        const double sig = vmax * fabs(dts) / (d == 0 ? G.dx : G.dy);
        if (!(sig < 0.999)) return false;
    }
    int xb, C;
    return pick_xy_shape(G, s, xb, C);
}

// One fused spatial stage src -> dst on the interior rows.  Ghost rows (FLUID sides) are not written here:
// api.cu runs the general x kernel on them (x sweeps update ghost rows, y sweeps never do, R16).
int launch_sweep_xy(vlasov_ctx* c, const Species& s, const double* src, double* dst, double dts, int xfirst) {
    const Geom& G = c->G;
    XYParams P;
    P.src = src; P.dst = dst;
    P.S = s.nvtot; P.row_stride = (long)G.nx * s.nvtot;
    P.nx = G.nx; P.ny = G.ny; P.g = G.g;
    P.nv1 = s.nv[1]; P.nv2 = s.nv[2];
    P.vminx = s.vmin[0]; P.dvx = s.dv[0]; P.vminy = s.vmin[1]; P.dvy = s.dv[1];
    P.kx = dts / G.dx; P.ky = dts / G.dy;
    P.finf = s.f_inf;
    P.bc_lo = G.bc_lo; P.bc_hi = G.bc_hi;
    int xb, C;
    if (!pick_xy_shape(G, s, xb, C)) return VLASOV_EINVAL;
    const int nblk = G.nx / xb;
    P.C = C;
    P.PC = C < s.nv[2] ? C : s.nv[2];
    const size_t smem = 128 + (xfirst ? 2 : 4) * (size_t)G.nx * C * 8;
    dim3 grid((unsigned)(s.nvtot / C));
    const int threads = nblk * C;
    const int lim = G.limiter ? 1 : 0;
    {
        Launch L(c, K_SWEEP_XY);
        if (xb == 8) { if (lim) launch_xy_t<8, 1>(P, xfirst, grid, threads, smem, c->stream); else launch_xy_t<8, 0>(P, xfirst, grid, threads, smem, c->stream); }
        else if (xb == 4) { if (lim) launch_xy_t<4, 1>(P, xfirst, grid, threads, smem, c->stream); else launch_xy_t<4, 0>(P, xfirst, grid, threads, smem, c->stream); }
        else { if (lim) launch_xy_t<1, 1>(P, xfirst, grid, threads, smem, c->stream); else launch_xy_t<1, 0>(P, xfirst, grid, threads, smem, c->stream); }
    }
    return cudaGetLastError() == cudaSuccess ? VLASOV_OK : VLASOV_ECUDA;
}

}  // namespace vl
