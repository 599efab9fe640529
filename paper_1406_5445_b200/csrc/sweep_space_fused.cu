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
//   * raw rows arrive by 2D tiled TMA into a ring of shared rows [x][c], several rows ahead of the compute;
//   * x couples threads: each thread reads its cells and the 3 halo cells of its x block from the shared row
//     (periodic wrap);
//   * y is private to a thread: a 2-row register window (the two arrays swap roles every row) plus the
//     previous flux per owned cell.
// Rows -2, -1 and ny, ny+1 are the boundary rows of the y sweep (R16, R19): periodic wrap, the wall
// image f(y_w + eta, vy) = f(y_w - eta, -vy), or FLUID ghost rows; they are loaded like any row.
#include <mutex>
#include <map>
#include <utility>
#include <type_traits>
#include "vlasov_internal.cuh"
#include "tma.cuh"

namespace vl {

struct XYParams {
    const double* __restrict__ src;
    double* __restrict__ dst;
    long S;            // doubles per spatial cell
    long row_stride;   // nx * S
    int nx, ny, g;
    int nyg;           // rows of a z slab (3D3V: blockIdx.y is the slab)
    int nv1, nv2;
    int nxb;           // x cells per TMA box (a box holds at most 256 rows: nx > 256 takes several boxes per row)
    int C;             // contiguous velocity cells per CTA
    int PC;            // cells per bulk copy (a piece of one v_z row, or the whole chunk)
    double vminx, dvx, vminy, dvy;
    double kx, ky;     // dts/dx, dts/dy
    double finf;
    int bc_lo, bc_hi;
};

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

// Can any of a batch of cells need its slopes limited?  High-word test of vlasov_internal.cuh, made once for the whole
// batch from running integer minima / maxima (conservative; comparisons, not differences of high words: for f < 0 or
// f > f_inf the high word of a bound is hugely negative):
//     every |d| of the batch  <  min( 2 min f, 2 (f_inf - max f) )   ==>   every eps of the batch is 1.
// hmin, hmax: signed min / max of the high words of the cells' values; dmax: max of the high words of |d| over every
// difference the batch uses.  One fp64 subtraction per batch (f_inf minus an upper bound of max f) instead of one per
// cell, 2 integer instructions per value instead of 6.
__device__ __forceinline__ bool batch_may_need(int hmin, int hmax, int dmax, double finf) {
    const double fmax_ub = __hiloint2double(hmax + 1, 0);          // > every value of the batch (f >= 0; else hmin < 0 decides)
    const int hb = min(hmin, __double2hiint(finf - fmax_ub)) + 0x00100000;
    return dmax >= hb;
}
__device__ __forceinline__ int hi_abs(double d) { return __double2hiint(d) & 0x7fffffff; }

// N partial fluxes alpha [ f0 + c1 eps+ d+ + c2 eps- d- ] of the cells q[1..N] of a line piece q[0..N+1]
// (q ordered in the direction of the flow, so eq. (47) is the same call on the reversed piece).
// The limiter test is batched: one vote per call, and the usual answer is "nobody".
// FULL: every lane of the warp makes this call together (the CTA-uniform copies of the row loop): votes with the full mask.
template <int N, int LIM, int FULL = 0>
__device__ __forceinline__ void flux_line(const double (&q)[N + 2], const Weights& W, double finf, double (&G)[N]) {
    double d[N + 1];
#pragma unroll
    for (int i = 0; i <= N; ++i) d[i] = q[i + 1] - q[i];
    if (LIM) {
        int hmin = __double2hiint(q[1]), hmax = hmin, dmax = hi_abs(d[0]);
#pragma unroll
        for (int i = 1; i <= N; ++i) {
            if (i < N) { hmin = min(hmin, __double2hiint(q[i + 1])); hmax = max(hmax, __double2hiint(q[i + 1])); }
            dmax = max(dmax, hi_abs(d[i]));
        }
        if (__any_sync(FULL ? 0xffffffffu : __activemask(), batch_may_need(hmin, hmax, dmax, finf))) {
#pragma unroll
            for (int i = 0; i < N; ++i) {
                double sp, sm;
                slopes_fast<1, FULL>(q[i], q[i + 1], q[i + 2], finf, sp, sm);
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
template <int XB, int CH, int LIM, int DIR, int FULL = 0>
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
    flux_line<CH + 1, LIM, FULL>(q, W, finf, G);         // fluxes out of positions 1+k CH .. 1+k CH+CH
    if (k > 0) G[0] = carry;
    carry = G[CH];
#pragma unroll
    for (int i = 0; i < CH; ++i) val[i] = q[i + 2] + (G[i] - G[i + 1]);
}

// x_chunk for a whole x block (CH = XB) whose own cells the thread still holds in registers (own[i] = cell ix0 + i, the
// y-swept values it has just written to the shared row): only the three halo cells are read from shared memory.
template <int XB, int LIM, int DIR, int FULL>
__device__ __forceinline__ void x_chunk_own(const double (&own)[XB], double (&val)[XB], unsigned sbuf, int ix0, int nx, int C8,
                                            unsigned cofs, const Weights& W, double finf) {
    double q[XB + 3], G[XB + 1];
#pragma unroll
    for (int p = 0; p < XB + 3; ++p) {
        if (p >= 2 && p < XB + 2) {
            q[p] = own[DIR > 0 ? p - 2 : XB + 1 - p];
        } else {
            int ix = DIR > 0 ? ix0 - 2 + p : ix0 + XB + 1 - p;
            if (ix < 0) ix += nx; else if (ix >= nx) ix -= nx;
            q[p] = lds(sbuf + ix * C8 + cofs);
        }
    }
    flux_line<XB + 1, LIM, FULL>(q, W, finf, G);
#pragma unroll
    for (int i = 0; i < XB; ++i) val[i] = q[i + 2] + (G[i] - G[i + 1]);
}

// NB steps of the y march at once (the owned cells of one x chunk): rows (r-2, r-1, r) = (ya, yb, gx) -> new average
// h of row r-1 (sigma_y >= 0, eq. 46) or r-2 (sigma_y < 0, eq. 47 on the mirrored line).  One limiter vote for all
// NB of them, so that the flux evaluations are independent instruction streams.
// ydmax: max high word of |row r-1 - row r-2| over the batch, left by the previous row's call (where it was the upper
// difference): the lower differences of this row need no second look.
// YD: the direction of the y flow where the caller knows it at compile time (+1 / -1), 0: Wy.pos at run time.
template <int NB, int LIM, int YD = 0>
__device__ __forceinline__ void y_batch(const double (&ya)[NB], const double (&yb)[NB], double (&yG)[NB],
                                        const double (&gx)[NB], const Weights& Wy, double finf, double (&h)[NB], int& ydmax) {
    const bool ypos = YD == 0 ? Wy.pos : YD > 0;
    double dlo[NB], dhi[NB];
    int hmin = 0x7fffffff, hmax = (int)0x80000000, dup = 0;
#pragma unroll
    for (int i = 0; i < NB; ++i) {
        dlo[i] = yb[i] - ya[i]; dhi[i] = gx[i] - yb[i];
        if (LIM) { hmin = min(hmin, __double2hiint(yb[i])); hmax = max(hmax, __double2hiint(yb[i])); dup = max(dup, hi_abs(dhi[i])); }
    }
    constexpr int FULL = YD != 0 ? 1 : 0;          // a known direction means a CTA-uniform copy of the row loop: whole warps
    const bool slow = LIM && __any_sync(FULL ? 0xffffffffu : __activemask(), batch_may_need(hmin, hmax, max(dup, ydmax), finf));
    ydmax = dup;
#pragma unroll
    for (int i = 0; i < NB; ++i) {
        double sp = ypos ? dhi[i] : -dlo[i], sm = ypos ? dlo[i] : -dhi[i];
        if (slow) { if (ypos) slopes_fast<1, FULL>(ya[i], yb[i], gx[i], finf, sp, sm); else slopes_fast<1, FULL>(gx[i], yb[i], ya[i], finf, sp, sm); }
        const double Gn = fma(Wy.w2, sm, fma(Wy.w1, sp, Wy.w0 * yb[i]));
        h[i] = ypos ? yb[i] + (yG[i] - Gn) : ya[i] + (Gn - yG[i]);
        yG[i] = Gn;
    }
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
// Shared memory: [NS mbarriers][NS raw rows]([2 y-swept rows] if !XFIRST).  Raw rows arrive by tiled TMA, NS - 1
// rows ahead of the row being worked on.
constexpr int XY_NS = 5;

constexpr int xy_default_chunk(int sp) { return sp > 0 ? 2048 / (sp > 0 ? sp : 1) : 0; }

// SP > 0: nx = SP spatial cells per row, NV^3 velocity cells, KC = the launcher's chunk for that shape (one piece:
// C = PC = KC): every stride of the kernel is a compile-time constant.  SP = 0: any shape, at run time.
template <int XB, int LIM, int XFIRST, int SP, int NV = 32, int KC = xy_default_chunk(SP)>
#ifndef VL_XY_MAXT
#define VL_XY_MAXT 512
#endif
#ifndef VL_XY_MINB
#define VL_XY_MINB 1
#endif
#ifndef VL_XY_CH
#define VL_XY_CH 4
#endif
#ifndef VL_XY_UNIDIR
#define VL_XY_UNIDIR 1
#endif
#ifndef VL_XY_OWN
#define VL_XY_OWN 1
#endif
__global__ void __launch_bounds__(VL_XY_MAXT, VL_XY_MINB) sweep_xy_kernel(const __grid_constant__ CUtensorMap tmap, XYParams P) {
    extern __shared__ __align__(128) unsigned char smraw[];
    constexpr long KS = (long)NV * NV * NV;
    if (SP && (P.nx != SP || P.C != KC || P.PC != KC || P.nv1 != NV || P.nv2 != NV || P.S != KS)) return;
    const int nx = SP ? SP : P.nx, nv1 = SP ? NV : P.nv1, nv2 = SP ? NV : P.nv2;
    const long S = SP ? KS : P.S, row_stride = SP ? (long)SP * KS : P.row_stride;
    const int C = SP ? KC : P.C, C8 = C * 8;
    const int c = threadIdx.x % C, blk = threadIdx.x / C;
    const int ix0 = blk * XB;
    const long v0 = (long)blockIdx.x * C;
    const long v = v0 + c;
    const int ivx = (int)(v / ((long)nv1 * nv2));
    const int ivy = (int)((v / nv2) % nv1);
    // the six weights of a velocity cell live in shared memory (wt[k][c]): 12 registers less per thread; only
    // the two flow directions stay in registers
    double* wt = reinterpret_cast<double*>(smraw + 128);
    bool xpos, ypos;
    {
        Weights W0x, W0y;
        W0x.set((P.vminx + (ivx + 0.5) * P.dvx) * P.kx);
        W0y.set((P.vminy + (ivy + 0.5) * P.dvy) * P.ky);
        xpos = W0x.pos; ypos = W0y.pos;
        if (blk == 0) {
            wt[0 * C + c] = W0x.w0; wt[1 * C + c] = W0x.w1; wt[2 * C + c] = W0x.w2;
            wt[3 * C + c] = W0y.w0; wt[4 * C + c] = W0y.w1; wt[5 * C + c] = W0y.w2;
        }
    }
    const unsigned bar0 = smem_addr(smraw);
    // a row buffer is made of C / PC pieces, each a dense [x][PC] TMA box (128-byte aligned)
    const int PC = SP ? KC : P.PC, npp = C / PC, X8 = PC * 8;
    const unsigned piecebytes = ((unsigned)nx * X8 + 127u) & ~127u;
    const unsigned rowbytes = piecebytes * npp;
    const unsigned raw0 = bar0 + 128 + ((6 * C * 8 + 127) & ~127);
    const unsigned hb0 = raw0 + XY_NS * rowbytes;
    const unsigned cofs = (unsigned)(c / PC) * piecebytes + (unsigned)(c % PC) * 8;
    const unsigned own = (unsigned)ix0 * X8 + cofs;
    const double finf = P.finf;

    // producer: thread 0 issues one tiled TMA load per piece and row (a piece = PC contiguous cells of every x:
    // a v_z row or a part of one, so that its wall image, i_vy mirrored (R19), is one box too)
    auto issue_row = [&](int r, int stage) {
        if (threadIdx.x == 0) {
            const unsigned bar = bar0 + 8 * stage;
            mbar_expect_tx(bar, (unsigned)nx * C8);
            bool m; const int ar = virtual_row(P, r, m);
            for (int p = 0; p < npp; ++p) {
                long vp = v0 + (long)p * PC;
                if (m) vp += (long)(nv1 - 1 - 2 * (int)((vp / nv2) % nv1)) * nv2;
                const int nxb = SP ? SP : P.nxb;
                for (int b = 0; b * nxb < nx; ++b)
                    tma_g2s_2d(raw0 + stage * rowbytes + p * piecebytes + (unsigned)(b * nxb) * X8, &tmap, (int)vp,
                               (ar + (int)blockIdx.y * P.nyg) * nx + b * nxb, bar);
            }
        }
    };
    if (threadIdx.x == 0) {
        for (int i = 0; i < XY_NS; ++i) mbar_init(bar0 + 8 * i, 1);
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    __syncthreads();
    // a barrier's phase cannot complete before thread 0's arrive.expect_tx, whatever order the copies land in
    const int rlast = P.ny + 1;
    for (int i = 0; i < XY_NS - 1; ++i) if (-2 + i <= rlast) issue_row(-2 + i, i);

    // y window of the owned cells: rows r-2 and r-1 sit in A and B, swapping roles every row (no moves)
    double A[XB], B[XB], yG[XB];
#pragma unroll
    for (int i = 0; i < XB; ++i) { A[i] = 0.0; B[i] = 0.0; yG[i] = 0.0; }
    const int orow_shift = ypos ? 1 : 2;
    constexpr int CH = XB < VL_XY_CH ? XB : VL_XY_CH;
    int ydm[XB / CH];                              // limiter test of the y march: see y_batch
#pragma unroll
    for (int i = 0; i < XB / CH; ++i) ydm[i] = 0;

    // one row; PAR = parity of r + 2: rows (r-2, r-1) = (A, B) if PAR == 0 else (B, A); the new row replaces r-2
    // XD, YD: the flow directions as compile-time constants (+1 / -1) where the whole CTA shares them, 0: per thread
#ifndef VL_XY_WREG
#define VL_XY_WREG 1
#endif
    double rw[6];
    {
        Weights W0x, W0y;
        W0x.set((P.vminx + (ivx + 0.5) * P.dvx) * P.kx);
        W0y.set((P.vminy + (ivy + 0.5) * P.dvy) * P.ky);
        rw[0] = W0x.w0; rw[1] = W0x.w1; rw[2] = W0x.w2; rw[3] = W0y.w0; rw[4] = W0y.w1; rw[5] = W0y.w2;
    }
    auto row = [&](auto par, auto xd, auto yd, int r, int stage, unsigned phase) {
        constexpr int PAR = decltype(par)::value, XD = decltype(xd)::value, YD = decltype(yd)::value;
        Weights Wx, Wy;
#if VL_XY_WREG
        if (XD != 0) {       // the CTA-uniform copies have the registers to keep the six weights (98 of 128)
            Wx.w0 = rw[0]; Wx.w1 = rw[1]; Wx.w2 = rw[2]; Wy.w0 = rw[3]; Wy.w1 = rw[4]; Wy.w2 = rw[5];
        } else
#endif
        {
            Wx.w0 = wt[0 * C + c]; Wx.w1 = wt[1 * C + c]; Wx.w2 = wt[2 * C + c];
            Wy.w0 = wt[3 * C + c]; Wy.w1 = wt[4 * C + c]; Wy.w2 = wt[5 * C + c];
        }
        Wx.pos = XD == 0 ? xpos : XD > 0;
        Wy.pos = YD == 0 ? ypos : YD > 0;
        const unsigned sraw = raw0 + stage * rowbytes;
        mbar_wait(bar0 + 8 * stage, phase);
        const int orow = r - orow_shift;
        double* po = P.dst + (long)(P.g + orow + (int)blockIdx.y * P.nyg) * row_stride + (long)ix0 * S + v;
        const bool store = orow >= 0 && orow < P.ny;
        const int nstage = stage == 0 ? XY_NS - 1 : stage - 1;      // stage of row r + NS - 1 = stage of row r - 1
        if (XFIRST) {
            // row r - 1 was left by every thread before the __syncthreads that ended it: refill its stage
            if (r + XY_NS - 1 <= rlast) issue_row(r + XY_NS - 1, nstage);
            double carry = 0.0;
#pragma unroll
            for (int k = 0; k < XB / CH; ++k) {
                double gx[CH];
                if (XD > 0 || (XD == 0 && Wx.pos)) {
                    x_chunk<XB, CH, LIM, 1, (XD != 0)>(k, carry, gx, sraw, ix0, nx, X8, cofs, Wx, finf);
                    double ya[CH], yb[CH], g[CH], h[CH];
#pragma unroll
                    for (int i = 0; i < CH; ++i) { const int it = k * CH + i; ya[i] = PAR == 0 ? A[it] : B[it]; yb[i] = PAR == 0 ? B[it] : A[it]; g[i] = yG[it]; }
                    y_batch<CH, LIM, YD>(ya, yb, g, gx, Wy, finf, h, ydm[k]);
#pragma unroll
                    for (int i = 0; i < CH; ++i) {
                        const int it = k * CH + i;
                        yG[it] = g[i];
                        if (PAR == 0) A[it] = gx[i]; else B[it] = gx[i];
                        if (store) __stcs(po + (long)it * S, h[i]);
                    }
                } else {
                    x_chunk<XB, CH, LIM, -1, (XD != 0)>(k, carry, gx, sraw, ix0, nx, X8, cofs, Wx, finf);
                    double ya[CH], yb[CH], g[CH], h[CH];
#pragma unroll
                    for (int i = 0; i < CH; ++i) { const int it = XB - 1 - (k * CH + i); ya[i] = PAR == 0 ? A[it] : B[it]; yb[i] = PAR == 0 ? B[it] : A[it]; g[i] = yG[it]; }
                    y_batch<CH, LIM, YD>(ya, yb, g, gx, Wy, finf, h, ydm[k]);
#pragma unroll
                    for (int i = 0; i < CH; ++i) {
                        const int it = XB - 1 - (k * CH + i);
                        yG[it] = g[i];
                        if (PAR == 0) A[it] = gx[i]; else B[it] = gx[i];
                        if (store) __stcs(po + (long)it * S, h[i]);
                    }
                }
            }
            __syncthreads();                       // everybody is done reading raw row r
        } else {
            const unsigned sh = hb0 + (unsigned)PAR * rowbytes;
            double h[XB];
            {
                double gx[XB];
#pragma unroll
                for (int i = 0; i < XB; ++i) gx[i] = lds(sraw + own + i * X8);
                if (PAR == 0) y_batch<XB, LIM, YD>(A, B, yG, gx, Wy, finf, h, ydm[0]); else y_batch<XB, LIM, YD>(B, A, yG, gx, Wy, finf, h, ydm[0]);
#pragma unroll
                for (int i = 0; i < XB; ++i) {
                    if (PAR == 0) A[i] = gx[i]; else B[i] = gx[i];
                    sts(sh + own + i * X8, h[i]);
                }
            }
            __syncthreads();                       // y-swept row complete; raw rows up to r are free
            if (r + XY_NS <= rlast) issue_row(r + XY_NS, stage);
            double carry = 0.0;
            if constexpr (VL_XY_OWN && XB == CH && XD != 0) {
                double o[XB];
                x_chunk_own<XB, LIM, XD, 1>(h, o, sh, ix0, nx, X8, cofs, Wx, finf);
                if (store) {
#pragma unroll
                    for (int i = 0; i < XB; ++i) __stcs(po + (long)(XD > 0 ? i : XB - 1 - i) * S, o[i]);
                }
            } else {
#pragma unroll
            for (int k = 0; k < XB / CH; ++k) {
                double o[CH];
                if (XD > 0 || (XD == 0 && Wx.pos)) {
                    x_chunk<XB, CH, LIM, 1, (XD != 0)>(k, carry, o, sh, ix0, nx, X8, cofs, Wx, finf);
                    if (store) {
#pragma unroll
                        for (int i = 0; i < CH; ++i) __stcs(po + (long)(k * CH + i) * S, o[i]);
                    }
                } else {
                    x_chunk<XB, CH, LIM, -1, (XD != 0)>(k, carry, o, sh, ix0, nx, X8, cofs, Wx, finf);
                    if (store) {
#pragma unroll
                        for (int i = 0; i < CH; ++i) __stcs(po + (long)(XB - 1 - (k * CH + i)) * S, o[i]);
                    }
                }
            }
            }
        }
    };
    if (!XFIRST) { if (XY_NS - 3 <= rlast) issue_row(-2 + XY_NS - 1, XY_NS - 1); }   // !XFIRST refills after its barrier: start one row deeper
    auto march = [&](auto xd, auto yd) {
        int stage = 0; unsigned phase = 0;
        for (int r = -2; r <= rlast; r += 2) {
            row(std::integral_constant<int, 0>{}, xd, yd, r, stage, phase);
            if (++stage == XY_NS) { stage = 0; phase ^= 1; }
            if (r + 1 <= rlast) {
                row(std::integral_constant<int, 1>{}, xd, yd, r + 1, stage, phase);
                if (++stage == XY_NS) { stage = 0; phase ^= 1; }
            }
        }
    };
    using P1 = std::integral_constant<int, 1>; using M1 = std::integral_constant<int, -1>; using R0 = std::integral_constant<int, 0>;
    // A CTA of a compile-time-shape kernel owns a piece of ONE v_z row (KC <= NV): v_x and v_y, and with them both flow
    // directions, are the same for all of its threads -- four copies of the row loop, each with its directions folded in
    // (no selects on the direction, no register moves where two branches meet); a CTA runs one of them.
    // (CTAs of 128 threads, five or more to an SM, would pull several copies through the instruction cache at once:
    // 24^3 with nx = 64 measured 4 % slower that way and keeps the per-thread directions)
    if (VL_XY_UNIDIR && SP > 0 && KC <= NV && (SP / XB) * KC >= 256) {
        if (xpos) { if (ypos) march(P1{}, P1{}); else march(P1{}, M1{}); }
        else { if (ypos) march(M1{}, P1{}); else march(M1{}, M1{}); }
    } else {
        march(R0{}, R0{});
    }
}

// The opt-in to more than 48 KiB of dynamic shared memory is a per-device function attribute and a MAXIMUM: it is raised
// when a launch needs more than any launch of that kernel on that device before it, never lowered.
template <class K>
static void ensure_smem_attr(K kernel, size_t smem) {
    static std::mutex mu;
    static std::map<std::pair<int, const void*>, size_t> granted;
    int dev = 0;
    cudaGetDevice(&dev);
    const auto key = std::make_pair(dev, (const void*)kernel);
    std::lock_guard<std::mutex> lock(mu);
    auto it = granted.find(key);
    if (it != granted.end() && it->second >= smem) return;
    cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    granted[key] = smem;
}

template <int XB, int LIM, int SP, int NV = 32, int KC = xy_default_chunk(SP)>
static void launch_xy_t(const CUtensorMap& tm, const XYParams& P, int xfirst, dim3 grid, int threads, size_t smem,
                        cudaStream_t st) {
    if (xfirst) {
        ensure_smem_attr(sweep_xy_kernel<XB, LIM, 1, SP, NV, KC>, smem);
        sweep_xy_kernel<XB, LIM, 1, SP, NV, KC><<<grid, threads, smem, st>>>(tm, P);
    } else {
        ensure_smem_attr(sweep_xy_kernel<XB, LIM, 0, SP, NV, KC>, smem);
        sweep_xy_kernel<XB, LIM, 0, SP, NV, KC><<<grid, threads, smem, st>>>(tm, P);
    }
}

// Shared memory of the fused kernel: barriers, weight table, NS raw rows (+ 2 y-swept rows), each row made of
// 128-byte aligned pieces.
static size_t xy_smem_bytes(const Geom& G, const Species& s, int C, int xfirst) {
    const int pc = C < s.nv[2] ? C : s.nv[2];
    const size_t piece = ((size_t)G.nx * pc * 8 + 127) & ~(size_t)127;
    const size_t row = piece * (C / pc);
    return 128 + ((6 * (size_t)C * 8 + 127) & ~(size_t)127) + (xfirst ? XY_NS : XY_NS + 2) * row;
}

// x cells per TMA box: a box dimension is at most 256, so a row of nx > 256 cells arrives as nx / nxb equal boxes
static int xy_box_rows(int nx) {
    for (int k = 1; k <= 16; ++k) if (nx % k == 0 && nx / k <= 256) return nx / k;
    return 0;
}

// Tile shape of the fused stage: XB x cells per thread, C contiguous velocity cells per CTA -- a power of two
// that divides the block, made of whole v_z rows or a part of one, at least 16 bytes, at most 512 threads.
static bool pick_xy_shape(const Geom& G, const Species& s, int& xb, int& C) {
    xb = 1;
    // 4 x cells per thread: 8 would halve the halo work but spills at the 128-register cap of 512 threads
    if (G.nx % 4 == 0) xb = 4;
    const int nblk = G.nx / xb;
    C = 32;
    // (a piece = min(cc, nv[2]) cells is one TMA box row: at least 16 bytes, so an odd nv[2] has no shape here)
    auto ok = [&](int cc) { return s.nvtot % cc == 0 && (s.nv[2] % cc == 0 || cc % s.nv[2] == 0) && s.nv[2] >= 2 && nblk * cc <= VL_XY_MAXT; };
    while (C >= 2 && !ok(C)) C >>= 1;
    if (C < 2) return false;
    if (xy_box_rows(G.nx) == 0) return false;      // no equal split of a row into TMA boxes of at most 256 x cells
    return xy_smem_bytes(G, s, C, 0) <= 200 * 1024;
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
    P.nx = G.nx; P.ny = G.ny; P.g = G.g; P.nyg = G.nyg;
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
    const size_t smem = xy_smem_bytes(G, s, C, xfirst);
    CUtensorMap tm;
    P.nxb = xy_box_rows(G.nx);
    if (!make_tensor_map_2d(&tm, src, s.nvtot, (long)G.nrows * G.nx, P.PC, P.nxb)) return VLASOV_ECUDA;
    dim3 grid((unsigned)(s.nvtot / C), (unsigned)G.nz);
    const int threads = nblk * C;
    const int lim = G.limiter ? 1 : 0;
    {
        Launch L(c, xfirst ? K_SWEEP_XY : K_SWEEP_YX);
        const bool v32 = s.nv[0] == 32 && s.nv[1] == 32 && s.nv[2] == 32 && xb == 4 && P.PC == C;
        const int cube = (s.nv[0] == s.nv[1] && s.nv[1] == s.nv[2] && xb == 4 && P.PC == C) ? s.nv[0] : 0;
        // the other shapes of BASELINE.json's configs 4 and 5
        if (cube == 24 && G.nx == 64 && C == 8) { if (lim) launch_xy_t<4, 1, 64, 24, 8>(tm, P, xfirst, grid, threads, smem, c->stream); else launch_xy_t<4, 0, 64, 24, 8>(tm, P, xfirst, grid, threads, smem, c->stream); }
        else if (cube == 48 && G.nx == 64 && C == 16) { if (lim) launch_xy_t<4, 1, 64, 48, 16>(tm, P, xfirst, grid, threads, smem, c->stream); else launch_xy_t<4, 0, 64, 48, 16>(tm, P, xfirst, grid, threads, smem, c->stream); }
        else if (cube == 40 && G.nx == 256 && C == 8) { if (lim) launch_xy_t<4, 1, 256, 40, 8>(tm, P, xfirst, grid, threads, smem, c->stream); else launch_xy_t<4, 0, 256, 40, 8>(tm, P, xfirst, grid, threads, smem, c->stream); }
        else
        if (v32 && G.nx == 128 && C == 8) { if (lim) launch_xy_t<4, 1, 128, 32, 8>(tm, P, xfirst, grid, threads, smem, c->stream); else launch_xy_t<4, 0, 128, 32, 8>(tm, P, xfirst, grid, threads, smem, c->stream); }
        else if (v32 && G.nx == 128 && C == 16) { if (lim) launch_xy_t<4, 1, 128>(tm, P, xfirst, grid, threads, smem, c->stream); else launch_xy_t<4, 0, 128>(tm, P, xfirst, grid, threads, smem, c->stream); }
        else if (v32 && G.nx == 32 && C == 32) { if (lim) launch_xy_t<4, 1, 32, 32, 32>(tm, P, xfirst, grid, threads, smem, c->stream); else launch_xy_t<4, 0, 32, 32, 32>(tm, P, xfirst, grid, threads, smem, c->stream); }
        else if (v32 && G.nx == 64 && C == 32) { if (lim) launch_xy_t<4, 1, 64>(tm, P, xfirst, grid, threads, smem, c->stream); else launch_xy_t<4, 0, 64>(tm, P, xfirst, grid, threads, smem, c->stream); }
        else if (xb == 4) { if (lim) launch_xy_t<4, 1, 0>(tm, P, xfirst, grid, threads, smem, c->stream); else launch_xy_t<4, 0, 0>(tm, P, xfirst, grid, threads, smem, c->stream); }
        else { if (lim) launch_xy_t<1, 1, 0>(tm, P, xfirst, grid, threads, smem, c->stream); else launch_xy_t<1, 0, 0>(tm, P, xfirst, grid, threads, smem, c->stream); }
    }
    return cudaGetLastError() == cudaSuccess ? VLASOV_OK : VLASOV_ECUDA;
}

}  // namespace vl
