// Velocity sweeps by backsubstitution (eqs. 33-35) and the table that drives them.
//
// The foot of the characteristic that ends on a face is affine in (face, transverse centre 1,
// transverse centre 2) for all three sweeps (eqs. 35, 34, 33 with the half kicks of eq. 26, R10), so
// per spatial cell the shift of face k of the line (k1, k2) is
//     sigma = c0 + c1 k + c2 k1 + c3 k2.
// A tiny kernel fills that table from E, B (a3); the ghost fill (section 4.2, eq. 63) writes the same
// table with its own affine map, so one set of sweep kernels serves both.
//
// Sweep kernels: the tile of lines is staged in shared memory (tiled TMA for the compile-time shapes, cp.async
// otherwise) between zero pad cells (f = 0 outside the box, R7), and ONE THREAD WALKS A SEGMENT of about 8 cells of
// one line: flux of eqs. (46)/(47) per face, eq. (38) per cell, zero flux through the two box faces.  Three walks,
// picked per warp by vote: march_seg_small (|sigma| < 1: the cells of the segment
// live in registers), march_seg_lite (shifts of several cells, sign changes: shift identity, no whole-cell sums),
// and the general per-face walk of march_cells.  vx: tile = all i_vx x 128 contiguous (i_vy,i_vz) cells, results
// straight to global memory.  vy+vz fused: tile = a few contiguous i_vx planes, vy: staging -> Bf, vz: Bf -> A,
// A -> global.  In place on f.
#include <map>
#include <mutex>
#include <tuple>
#include <type_traits>
#include "vlasov_internal.cuh"
#include "tma.cuh"

namespace vl {

// ------------------------------------------------------------------------------------------------
// a3: fields at the cell centre (R17) and the Lorentz sweep table
// ------------------------------------------------------------------------------------------------
struct TableParams {
    const double* __restrict__ E;
    const double* __restrict__ B;
    double* __restrict__ table;
    int nx, nyg, nz, fields_yee, wall;
    double qm_half_dt;        // (q/m)(dt/2), eqs. (26), (28)
    double vmin[3], dv[3];
    double finf;
    int* err;
};

__global__ void lorentz_table_kernel(TableParams P) {
    const int cell = blockIdx.x * blockDim.x + threadIdx.x;
    const int ncell = P.nx * P.nyg * P.nz;
    if (cell >= ncell) return;
    const int ix = cell % P.nx, j = (cell / P.nx) % P.nyg, k = cell / (P.nx * P.nyg);
    const long PL = (long)ncell;
    double Ec[3], Bc[3];
    if (!P.fields_yee) {
        for (int d = 0; d < 3; ++d) { Ec[d] = P.E[d * PL + cell]; Bc[d] = P.B[d * PL + cell]; }
    } else {
        // cell (i,j,k) spans [i dx,(i+1)dx] x [j dy,(j+1)dy] x [k dz,(k+1)dz]; Ex(i+1/2,j,k) Ey(i,j+1/2,k) Ez(i,j,k+1/2)
        // Bx(i,j+1/2,k+1/2) By(i+1/2,j,k+1/2) Bz(i+1/2,j+1/2,k) (R17 / R24): linear interpolation to the centre.
        // With nz = 1 the z neighbour is the cell itself and the sums below are the 2D ones bit for bit.
        const int ip = (ix + 1) % P.nx, kp = (k + 1) % P.nz;
        int jp = j + 1;
        double up = 1.0;
        if (jp >= P.nyg) { jp = 0; if (P.wall) up = 0.0; }
        auto at = [&](const double* A, int d, int kk, int jj, int ii) { return A[d * PL + ((long)kk * P.nyg + jj) * P.nx + ii]; };
        Ec[0] = 0.25 * ((at(P.E, 0, k, j, ix) + up * at(P.E, 0, k, jp, ix)) + (at(P.E, 0, kp, j, ix) + up * at(P.E, 0, kp, jp, ix)));
        Ec[1] = 0.25 * ((at(P.E, 1, k, j, ix) + at(P.E, 1, k, j, ip)) + (at(P.E, 1, kp, j, ix) + at(P.E, 1, kp, j, ip)));
        Ec[2] = 0.25 * (at(P.E, 2, k, j, ix) + at(P.E, 2, k, j, ip) + up * at(P.E, 2, k, jp, ix) + up * at(P.E, 2, k, jp, ip));
        Bc[0] = 0.5 * (at(P.B, 0, k, j, ix) + at(P.B, 0, k, j, ip));
        Bc[1] = 0.5 * (at(P.B, 1, k, j, ix) + up * at(P.B, 1, k, jp, ix));
        Bc[2] = 0.5 * (at(P.B, 2, k, j, ix) + at(P.B, 2, kp, j, ix));
    }
    // eq. (28): t = (q/m)(dt/2) B, s = 2t/(1+t^2); eq. (26): h = (q/m)(dt/2) E
    const double tx = P.qm_half_dt * Bc[0], ty = P.qm_half_dt * Bc[1], tz = P.qm_half_dt * Bc[2];
    const double hx = P.qm_half_dt * Ec[0], hy = P.qm_half_dt * Ec[1], hz = P.qm_half_dt * Ec[2];
    const double den = 1.0 + (tx * tx + ty * ty + tz * tz);
    const double sx = 2.0 * tx / den, sy = 2.0 * ty / den, sz = 2.0 * tz / den;
    const double D1 = 1.0 - ty * sy - tz * sz;       // denominator of eq. (35)
    const double D2 = 1.0 - tx * sx - ty * sy;       // denominator of eq. (34)
    if (!(D1 > 0.0 && D2 > 0.0)) { atomicCAS(P.err, 0, VLASOV_EDOMAIN); }   // R13
    double* T = P.table + (long)cell * TAB;
    const double wx0 = P.vmin[0] + 0.5 * P.dv[0], wy0 = P.vmin[1] + 0.5 * P.dv[1], wz0 = P.vmin[2] + 0.5 * P.dv[2];
    {   // vx sweep, eq. (35): foot = ((a - hx) - (vy + hy) K1 - (vz + hz) K2)/D1 - hx
        const double iD = 1.0 / D1;
        const double K1 = tx * sy + sz, K2 = tx * sz - sy;
        const double om = -(ty * sy + tz * sz) * iD;                    // 1 - 1/D1
        const double idv = 1.0 / P.dv[0];
        T[0] = (P.vmin[0] * om + hx + hx * iD + (hy * K1 + hz * K2) * iD + (wy0 * K1 + wz0 * K2) * iD) * idv;
        T[1] = om;
        T[2] = P.dv[1] * K1 * iD * idv;
        T[3] = P.dv[2] * K2 * iD * idv;
    }
    {   // vy sweep, eq. (34): foot = (vx - hx) C1 + (b - hy) C2 + (vz + hz) g - hy
        const double g = (ty * sz - sx) / D2;
        const double C1 = sx * ty + sz - (tz * sx - sy) * g;
        const double omC2 = tx * sx + tz * sz + (tz * sy + sx) * g;     // 1 - C2
        const double C2 = 1.0 - omC2;
        const double idv = 1.0 / P.dv[1];
        T[4] = (P.vmin[1] * omC2 + hy * C2 + hy + hx * C1 - hz * g - wx0 * C1 - wz0 * g) * idv;
        T[5] = omC2;
        T[6] = -P.dv[0] * C1 * idv;
        T[7] = -P.dv[2] * g * idv;
    }
    {   // vz sweep, eq. (33): foot = (vx - hx) Z1 + (vy - hy) Z2 + (c - hz) Z3 - hz
        const double Z1 = tz * sx - sy, Z2 = tz * sy + sx;
        const double omZ3 = tx * sx + ty * sy;                          // 1 - Z3
        const double Z3 = 1.0 - omZ3;
        const double idv = 1.0 / P.dv[2];
        T[8] = (P.vmin[2] * omZ3 + hz * Z3 + hz + hx * Z1 + hy * Z2 - wx0 * Z1 - wy0 * Z2) * idv;
        T[9] = omZ3;
        T[10] = -P.dv[0] * Z1 * idv;
        T[11] = -P.dv[1] * Z2 * idv;
    }
    T[12] = P.finf; T[13] = P.finf; T[14] = P.finf;
    T[15] = 1.0;
    T[16] = (double)cell;
}

int launch_lorentz_table(vlasov_ctx* c, const Species& s, const double* E, const double* B, double dt) {
    TableParams P;
    P.E = E; P.B = B; P.table = c->table;
    P.nx = c->G.nx; P.nyg = c->G.nyg; P.nz = c->G.nz; P.fields_yee = c->G.fields_yee; P.wall = c->G.wall;
    P.qm_half_dt = (s.q / s.m) * (dt / 2.0);
    for (int d = 0; d < 3; ++d) { P.vmin[d] = s.vmin[d]; P.dv[d] = s.dv[d]; }
    P.finf = s.f_inf;
    P.err = c->errflag;
    const int ncell = P.nx * P.nyg * P.nz;
    {
        Launch L(c, K_TABLE);
        lorentz_table_kernel<<<(ncell + 127) / 128, 128, 0, c->stream>>>(P);
    }
    return cudaGetLastError() == cudaSuccess ? VLASOV_OK : VLASOV_ECUDA;
}

// The two weights of eq. (46) as functions of alpha = b: c1 = (1-b)(2-b)/6, c2 = (1-b)(1+b)/6.  Written so that no
// instruction has more than one constant operand (1 and 1/2 are immediates, 1/6 comes from the constant bank): with two,
// one of them has to be moved into registers again at every face (8 of the ~50 instructions of a face were such moves).
//   c2 = (1 - b^2) / 6,   c1 + c2 = (1 - b) / 2.
__device__ __forceinline__ void pfc_weights(double b, double& c1, double& c2) {
#ifdef VL_POLY_OLD
    const double b2 = b * b;
    c1 = fma(b2, 1.0 / 6.0, fma(b, -0.5, 1.0 / 3.0));
    c2 = fma(b2, -1.0 / 6.0, 1.0 / 6.0);
#else
    c2 = (1.0 - b * b) * (1.0 / 6.0);
    c1 = fma(1.0 - b, 0.5, -c2);
#endif
}

// Flux through face k (between cells k-1 and k, 1 <= k <= N-1) of a ZERO-PADDED line in shared memory:
// L = shared byte address of cell 0, st8 = stride in bytes, cells -3..-1 and N..N+2 hold zeros (f = 0
// outside the box, R7).  eq. (46) for sigma >= 0, eq. (47) (sum repaired, R5) for sigma < 0: the same
// expression on the mirrored line.  floor() by a round-down add of 1.5 * 2^52: n sits in the low word,
// alpha = |sigma| - n in [0,1).
template <int LIM>
__device__ __forceinline__ double face_flux_pad(unsigned L, int st8, int N, int k, double sigma, double finf) {
    const double M = 6755399441055744.0;
    const double as = fabs(sigma);
    const double r = __dadd_rd(as, M);
    const int n = __double2loint(r);
    const double b = as - (r - M);
    const int sg = __double2hiint(sigma) >> 31;      // 0: sigma >= 0, -1: sigma < 0
    int j = k + (n ^ ~sg);                           // foot cell: k-1-n | k+n
    double sum = 0.0;
    if (n > 0) {                                     // the n whole cells between foot cell and face
        const int m0 = k - (n & ~sg);                // k-n | k
        const int lo = max(m0, 0), hi = min(m0 + n, N);
        unsigned am = L + lo * st8;
#pragma unroll 1
        for (int m = lo; m < hi; ++m) { sum += lds(am); am += st8; }
    }
    j = min(max(j, -2), N + 1);
    const unsigned aj = L + j * st8;
    const int ust8 = (st8 ^ sg) - sg;                // +st8 | -st8
    const double f0 = lds(aj);
    const double fm = lds(aj - ust8);
    const double fp = lds(aj + ust8);
    double sp, sm;
    slopes_fast<LIM>(fm, f0, fp, finf, sp, sm);
    // alpha [ f0 + (1-a)(2-a)/6 sp + (1-a)(1+a)/6 sm ]: the two weights as polynomials in alpha
    double c1, c2;
    pfc_weights(b, c1, c2);
    const double phi = fma(b, fma(c1, sp, fma(c2, sm, f0)), sum);
    // phi for sigma >= 0, -phi otherwise: flip the sign bit with sigma's
    return __hiloint2double(__double2hiint(phi) ^ (sg & 0x80000000), __double2loint(phi));
}

// Zero cells on either side of every line of a tile (f = 0 outside the box, R7): the general walk clamps the foot to
// [-2, N+1] and reads its two neighbours, the register-window walk reads cells -2 .. N+1.
constexpr int V_PAD = 3;
// Faces per limiter vote of the register-window walk (march_seg_small).  The vx kernel has registers to spare (2 CTAs
// per SM): 3 faces per vote give it three independent flux evaluations between votes.  The vy+vz kernel runs 3 CTAs
// per SM at 80 registers, where batches spill: one face per vote (measured, profiles/README.md).
#ifndef VL_X_BATCH
#define VL_X_BATCH 3
#endif
#ifndef VL_YZ_BATCH
#define VL_YZ_BATCH 1
#endif
#ifndef VL_YZ_MINB
#define VL_YZ_MINB 3
#endif
#ifndef VL_LITE_PEEL
#define VL_LITE_PEEL 1
#endif
// faces per trip of the lite walk's rolled loop: 4 for the 32x32 vy+vz kernel (2.90 -> 2.85 ms per cycle of config 3), 2
// elsewhere (4 measured 5 % slower on 48x48 planes, 8 misses the instruction cache: 1.41 -> 1.62 ms on nv32)
#ifndef VL_LITE_UNROLL
#define VL_LITE_UNROLL 2
#endif
#ifndef VL_LITE_UNROLL32
#define VL_LITE_UNROLL32 4
#endif

struct OutShared {       // cells of a line in shared memory: cell0 = byte address of cell a
    unsigned a; int st8;
    __device__ __forceinline__ void put(double v) { sts(a, v); a += st8; }
    __device__ __forceinline__ void step(int dir) { st8 *= dir; }
    __device__ __forceinline__ void skip(int n) { a += n * st8; }
};
struct OutGlobal {       // cells of a line in global memory (streaming store)
    double* p; long st;
    __device__ __forceinline__ void put(double v) { __stcs(p, v); p += st; }
    __device__ __forceinline__ void step(int dir) { st *= dir; }
    __device__ __forceinline__ void skip(int n) { p += n * st; }
};

// Segment of SEG cells [a, a+SEG) whose SEG+1 faces all have |sigma| < 1 (no whole cells in eqs. 46/47) and one
// flow direction: the SEG+3 cells the fluxes touch are read ONCE into registers, in the direction of the flow
// (eq. 47 = eq. 46 on the mirrored line), and face m of the walk takes (q[m], q[m+1], q[m+2]).  About a
// quarter of the instructions of the general walk below.
//   walk position i <-> cell a-2+i (sigma >= 0) | a+SEG+1-i (sigma < 0);  face m <-> face a+m | a+SEG-m.
template <int SEG, int LIM, int FULL, int NB, class Out>
__device__ __forceinline__ void march_seg_small(unsigned L, int st8, int N, int a, double sig_a, double sig_b,
                                                double s1, double finf, Out out) {
    const bool pos = !(sig_a < 0.0 || sig_b < 0.0);      // the caller made sure the two do not disagree
    const int dir = pos ? 1 : -1;
    const int ust8 = pos ? st8 : -st8;
    unsigned addr = L + (pos ? a - 2 : a + SEG + 1) * st8;
    double q[SEG + 3];
#pragma unroll
    for (int i = 0; i < SEG + 3; ++i) { q[i] = lds(addr); addr += ust8; }
    // box faces carry no flux (R7): the first / last face of the walk may be one
    const bool zero_first = pos ? a == 0 : a + SEG == N;
    const bool zero_last = pos ? a + SEG == N : a == 0;
    double sig = pos ? sig_a : sig_b;
    const double ds = pos ? s1 : -s1;
    if (!pos) { out.skip(SEG - 1); }
    out.step(dir);
    double Gp = 0.0;
    if constexpr (NB == 1) {
        // one limiter vote per face (slopes_fast): the leanest form in registers, for the kernel that has none to spare
#pragma unroll
        for (int m = 0; m <= SEG; ++m) {
            double sp, sm;
            slopes_fast<LIM, FULL>(q[m], q[m + 1], q[m + 2], finf, sp, sm);
            const double bq = fabs(sig);
            double c1, c2;
            pfc_weights(bq, c1, c2);
            double G = bq * fma(c1, sp, fma(c2, sm, q[m + 1]));
            if ((m == 0 && zero_first) || (m == SEG && zero_last)) G = 0.0;
            if (m > 0) out.put(q[m + 1] + (Gp - G));     // eq. (38) for the cell between walk faces m-1 and m
            Gp = G;
            sig += ds;
        }
    } else
    // NB faces at a time: ONE limiter vote per batch (all lanes sit on the same faces), so that the NB flux
    // evaluations are independent instruction streams between the votes
#pragma unroll
    for (int m0 = 0; m0 <= SEG; m0 += NB) {
        double sp[NB], sm[NB];
        bool need = false, needB = false;
        // High-word test of slopes_fast, once for the batch (conservative): every |d| of the batch below
        // min(2 min f, 2 (f_inf - max f)) means every eps is 1.  Running integer min / max of the high words, one fp64
        // subtraction per batch; comparisons, not differences (the high word of a bound is hugely negative for f < 0
        // or f > f_inf: round-off leaves -1e-17 behind).
        int hmin = 0x7fffffff, hmx = (int)0x80000000, dmax = LIM ? (__double2hiint(q[m0 + 1] - q[m0]) & 0x7fffffff) : 0;
#pragma unroll
        for (int i = 0; i < NB; ++i) {
            const int m = m0 + i;
            if (m > SEG) break;
            const double f0 = q[m + 1];
            sp[i] = q[m + 2] - f0; sm[i] = f0 - q[m];
            if (LIM) {
                hmin = min(hmin, __double2hiint(f0)); hmx = max(hmx, __double2hiint(f0));
                dmax = max(dmax, __double2hiint(sp[i]) & 0x7fffffff);
            }
        }
        if (LIM) {
            const int hg = __double2hiint(finf - __hiloint2double(hmx + 1, 0)) + 0x00100000;
            need = dmax >= min(hmin + 0x00100000, hg);
            needB = dmax >= hg;
        }
        // (without FULL the lanes voting together are whoever is here right now: the votes only decide which of two
        // equivalent evaluations runs, so any grouping that includes the lane itself is right)
        if (LIM && __any_sync(FULL ? 0xffffffffu : __activemask(), need)) {
            if (!__any_sync(FULL ? 0xffffffffu : __activemask(), needB)) {
                // only the positivity bound 2 f0 can bind: eps+ d+ = min(d+, hiA), eps- d- = max(d-, -hiA)
#pragma unroll
                for (int i = 0; i < NB; ++i) {
                    if (m0 + i > SEG) break;
                    const double hiA = relu_bits(q[m0 + i + 1] + q[m0 + i + 1]), nA = -hiA;
                    sp[i] = sp[i] < hiA ? sp[i] : hiA;
                    sm[i] = sm[i] > nA ? sm[i] : nA;
                }
            } else {
#pragma unroll
                for (int i = 0; i < NB; ++i) {
                    if (m0 + i > SEG) break;
                    slopes_exact(q[m0 + i + 1], finf, sp[i], sm[i]);
                }
            }
        }
#pragma unroll
        for (int i = 0; i < NB; ++i) {
            const int m = m0 + i;
            if (m > SEG) break;
            const double bq = fabs(sig);
            double c1, c2;
            pfc_weights(bq, c1, c2);
            double G = bq * fma(c1, sp[i], fma(c2, sm[i], q[m + 1]));
            if ((m == 0 && zero_first) || (m == SEG && zero_last)) G = 0.0;
            if (m > 0) out.put(q[m + 1] + (Gp - G));     // eq. (38) for the cell between walk faces m-1 and m
            Gp = G;
            sig += ds;
        }
    }
}

// Segment of SEG cells with shifts of any size whose lanes keep one flow direction along the segment (CROSS = 0), or
// change it once where |sigma| < 1 (CROSS = 1).  Walk in the direction of the flow as above, tau = |sigma| along it;
// nothing is kept in registers, a face reads the three cells around its foot.  Shift identity: with Phi = S + G
// (S the n whole cells of eqs. 46/47, G the partial cell) and n changing by at most one from face to face,
//     f_own + S_{m-1} - S_m  =  f0_m            n_m = n_{m-1}
//                            =  0               n_m = n_{m-1} + 1
//                            =  f0_m + fm_m     n_m = n_{m-1} - 1
// (f0_m, fm_m: foot cell of face m and its upstream neighbour, read for G_m anyway), so eq. (38) needs neither the
// whole-cell sums nor the cell itself.  A face against the flow (CROSS, n = 0 there) reads its foot one cell downstream,
// mirrored, and its own cell is fp.  The last face of the box carries no flux (R7): its S is added back, cell by cell.
//   flow cell c <-> cell a+c (sigma >= 0) | a+SEG-1-c (sigma < 0);  walk face m lies between flow cells m-1 and m.
template <int SEG, int LIM, int FULL, int CROSS, int LU, class Out>
__device__ __forceinline__ void march_seg_lite(unsigned L, int st8, int N, int a, double sig_a, double sig_b,
                                               double s1, double finf, Out out) {
    const double M = 6755399441055744.0;
    const bool pos = !(sig_a < 0.0 || sig_b < 0.0);
    const int u = pos ? st8 : -st8;
    unsigned fb = L + (pos ? a - 1 : a + SEG) * st8;     // flow cell m-1
    double tau = pos ? sig_a : -sig_b;                   // tau_m = tau_0 + m s1 in either direction
    const bool zero_first = pos ? a == 0 : a + SEG == N;
    const bool zero_last = pos ? a + SEG == N : a == 0;
    if (!pos) { out.skip(SEG - 1); }
    out.step(pos ? 1 : -1);
    double Gp = 0.0;
    int np = 0;
    // The first face only leaves its flux behind and is peeled off (its special cases cost five predicated instructions
    // at every face of a rolled loop); the other SEG faces run VL_LITE_UNROLL per trip of a rolled loop: the walks of a
    // sweep must share the 32 KB instruction cache.
    auto face = [&](int m, auto first_c) {
        constexpr bool FIRST = decltype(first_c)::value;
        const double at = fabs(tau);
        const double r = __dadd_rd(at, M);
        const int n = __double2loint(r);
        const double bq = at - (r - M);
        unsigned F = fb - n * u;                         // foot: flow cell m-1-n
        int uu = u;
        bool against = false;
        double bs = bq;                                  // bq with the sign of tau
        if (CROSS) {
            const int th = __double2hiint(tau);
            against = th < 0;
            F = against ? fb + u : F;                    // n = 0 there: foot = flow cell m, mirrored
            uu = against ? -u : u;
            bs = __hiloint2double(__double2hiint(bq) | (th & 0x80000000), __double2loint(bq));
        }
        const double f0 = lds(F), fm = lds(F - uu), fp = lds(F + uu);
        double sp, sm;
        slopes_fast<LIM, FULL>(fm, f0, fp, finf, sp, sm);
        double c1, c2;
        pfc_weights(bq, c1, c2);
        double G = bs * fma(c1, sp, fma(c2, sm, f0));
        if (FIRST) {
            if (zero_first) G = 0.0;
        } else {
            double T = f0;
            if (__any_sync(FULL ? 0xffffffffu : __activemask(), n != np)) {      // a quarter of the faces of a warp
                if (n > np) T = 0.0;
                if (n < np) T = f0 + fm;
            }
            if (CROSS && against) T = fp;
            if (m == SEG && zero_last) {
                G = 0.0;
                unsigned w = fb;
#pragma unroll 1
                for (int l = 0; l < n; ++l) { T += lds(w); w -= u; }
            }
            out.put(T + (Gp - G));
        }
        Gp = G;
        np = n;
        tau += s1;
        fb += u;
    };
#if VL_LITE_PEEL
    face(0, std::true_type{});
    constexpr int LITE_UNROLL = LU;
#pragma unroll LITE_UNROLL
    for (int m = 1; m <= SEG; ++m) face(m, std::false_type{});
#else
#pragma unroll 3
    for (int m = 0; m <= SEG; ++m) { if (m == 0) face(m, std::true_type{}); else face(m, std::false_type{}); }
#endif
}

// One thread remaps cells [a, b) of one line: flux per face, eq. (38) per cell.  sigma of face k is
// s0 + s1 k (accumulated).  out.put(value) stores the new average of the next cell (a, a+1, ...).
// FAST: 8-cell segments may take the flow-ordered walks (2: every lane of the warp is here).  LOOSE: the 4th cell
// before a line is readable memory (any value), which admits floor|sigma| = 2 at a box face.
// LU: faces per trip of the rolled loop of march_seg_lite (after its peeled first face).
// PAD: zero cells on either side of the line (V_PAD, or more where the caller's layout has them).
template <int LIM, int FAST, int LOOSE = 0, int NB = 1, int LU = VL_LITE_UNROLL, int PAD = V_PAD, class Out>
__device__ __forceinline__ void march_cells(unsigned L, int st8, int N, int a, int b, double s0, double s1,
                                            double finf, Out& out) {
    if (a >= b) return;                              // a trailing work item beyond the end of the line: nothing to do
    double sig = fma(s1, (double)a, s0);
    constexpr int SEG = 8;
    if (FAST && b - a == SEG) {
        // sigma is affine along the line: |sigma| < 1 and one sign at both end faces hold on every face between.
        const double sig_b = fma(s1, (double)b, s0);
        const bool cross = sig * sig_b < 0.0;
        const bool sub = fabs(sig) < 1.0 && fabs(sig_b) < 1.0;
        constexpr int FULL = FAST == 2 ? 1 : 0;        // FAST == 2: every lane of the warp is here
        const unsigned mask = FULL ? 0xffffffffu : __activemask();
        if (__all_sync(mask, sub && !cross)) {
            march_seg_small<SEG, LIM, FULL, NB>(L, st8, N, a, sig, sig_b, s1, finf, out);
            return;
        }
        // march_seg_lite: its first face reads flow cells -3-n .. -1-n, with PAD zero cells before the line; the
        // reads of a box face are discarded (zero flux), and n grows by less than 1/2 per face
        const bool pos = !(sig < 0.0 || sig_b < 0.0);
        const double t0 = pos ? sig : sig_b;
        const int dist = pos ? a : N - b;              // cells between the box face and the first face of the walk
        const double bound = (LOOSE && dist == 0) ? (double)PAD - 0.5 : (double)(min(dist, 32) + PAD - 1);
        const bool lite = fabs(t0) < bound && fabs(s1) <= 0.5 && (!cross || sub);
        if (__all_sync(mask, lite)) {
            if (__any_sync(mask, cross)) march_seg_lite<SEG, LIM, FULL, 1, LU>(L, st8, N, a, sig, sig_b, s1, finf, out);
            else march_seg_lite<SEG, LIM, FULL, 0, LU>(L, st8, N, a, sig, sig_b, s1, finf, out);
            return;
        }
    }
    double phi_lo = a > 0 ? face_flux_pad<LIM>(L, st8, N, a, sig, finf) : 0.0;
    unsigned ci = L + a * st8;
    const int bi = b < N ? b : N - 1;                // faces a+1 .. bi are interior
#pragma unroll 4
    for (int k = a + 1; k <= bi; ++k) {
        sig += s1;
        const double phi_hi = face_flux_pad<LIM>(L, st8, N, k, sig, finf);
        out.put(lds(ci) + (phi_lo - phi_hi));        // eq. (38): f + (Phi_{i-1/2} - Phi_{i+1/2})
        ci += st8;
        phi_lo = phi_hi;
    }
    if (b == N) out.put(lds(ci) + phi_lo);           // zero flux through the upper box face (R7)
}

struct VParams {
    const double* fsrc;   // what the vx sweep READS (== f: in place; the ping-pong buffer after a fused spatial stage)
    double* __restrict__ f;
    const double* __restrict__ table;
    long S;
    int nv0, nv1, nv2;
    int cell0;        // first spatial cell (ghost-inclusive linear index) of this launch
    int ct;           // columns per tile (vx kernel) / planes per tile (vyz kernel)
    int ntile;        // tiles per spatial cell
    int ntot;         // tiles of this launch
    int nseg;         // threads per line (vx kernel; vy lines of the vyz kernel)
    int nseg2;        // threads per vz line
    // moments fused into the vy+vz kernel (VXV order, NEXT-1): out[10][mom_ncell] of the cells of this launch, or null
    double* __restrict__ mom;
    int mom_ncell;
    double vmin[3], dv[3];
};

constexpr int V_THREADS = 256;

// ------------------------------------------------------------------------------------------------
// a4: vx sweep.  Tile = all i_vx x CT contiguous (i_vy,i_vz) columns, rows -V_PAD..-1 and N..N+V_PAD-1 zero.
// One thread marches a segment of one column; a warp reads/writes 256 contiguous bytes per step.
// Persistent: a CTA loops over tiles, the pad rows are zeroed once.
// ------------------------------------------------------------------------------------------------
// CN > 0: a CN^3 velocity block with the launcher's tile shape for it (128 columns, 2 segments), all compile-time.
template <int LIM, int CN>
__global__ void __launch_bounds__(V_THREADS, CN ? 3 : 4) vsweep_x_kernel(VParams P) {
    extern __shared__ double sm[];
    if (CN && (P.ct != 128 || P.nseg != CN / 8 || P.nv0 != CN || P.nv1 != CN || P.nv2 != CN)) return;
    const int CT = CN ? 128 : P.ct, N = CN ? CN : P.nv0, H = CT >> 1;
    const int nv2 = CN ? CN : P.nv2, nsegx = CN ? CN / 8 : P.nseg;
    const int plane = CN ? CN * CN : P.nv1 * P.nv2;
    const int ntile = CN ? (CN * CN + 127) / 128 : P.ntile;
    double* A = sm + V_PAD * CT;
    for (int e = threadIdx.x; e < V_PAD * CT; e += V_THREADS) { sm[e] = 0.0; A[N * CT + e] = 0.0; }
    const int seglen = (N + nsegx - 1) / nsegx;
    for (int tile = blockIdx.x; tile < P.ntot; tile += gridDim.x) {
        const int cell = P.cell0 + tile / ntile;
        const int c0 = (tile % ntile) * CT;
        const int ncol = min(CT, plane - c0);
        const double* T = P.table + (long)cell * TAB;
        const double t0 = T[0], t1 = T[1], t2 = T[2], t3 = T[3], finf = T[12], scale = T[15];
        const double* fsrc = P.fsrc + (long)T[16] * P.S + c0;
        double* fb = P.f + (long)cell * P.S + c0;
        if (CN || !(plane & 1)) {      // pairs of columns by 16-byte loads: every row of the tile starts on an even cell
            for (int e = threadIdx.x; e < N * H; e += V_THREADS) {
                const int k = e / H, c = 2 * (e - k * H);
                double2 v = make_double2(0.0, 0.0);
                if (c < ncol) { v = __ldcs(reinterpret_cast<const double2*>(fsrc + (long)k * plane + c)); v.x *= scale; v.y *= scale; }
                *reinterpret_cast<double2*>(A + k * CT + c) = v;
            }
        } else {                       // nv[1] nv[2] odd: column by column
            for (int e = threadIdx.x; e < N * CT; e += V_THREADS) {
                const int k = e / CT, c = e - k * CT;
                A[k * CT + c] = c < ncol ? __ldcs(fsrc + (long)k * plane + c) * scale : 0.0;
            }
        }
        __syncthreads();
        for (int wi = threadIdx.x; wi < CT * nsegx; wi += V_THREADS) {
            const int seg = wi / CT, c = wi - seg * CT;
            if (c < ncol) {
                const int col = c0 + c;
                const int k1 = col / nv2, k2 = col - k1 * nv2;
                const double s0 = t0 + t2 * k1 + t3 * k2;
                const int a = seg * seglen, b = min(a + seglen, N);
                OutGlobal o{fb + c + (long)a * plane, (long)plane};
                march_cells<LIM, (CN ? 1 : 0)>(smem_addr(A + c), CT * 8, N, a, b, s0, t1, finf, o);
            }
        }
        __syncthreads();
    }
}

// ------------------------------------------------------------------------------------------------
// a4 with the tiles prefetched: the same walk, but the tile of the NEXT two visits of this CTA is already on
// its way when a tile is worked on (2D tiled TMA, box {128 columns, CN rows}, one instruction per tile, two
// buffers + mbarriers).  The plain kernel above spends about 40 % of its stall samples waiting for its own
// global loads (profiles/).  CN^3 blocks with CN^2 a multiple of 128; not for the ghost fill (its tiles read
// another cell and are scaled).  Shared memory, in rows of 128 doubles:
//   [V_PAD zero rows][CN rows, buffer 0][V_PAD zero rows][CN rows, buffer 1][V_PAD zero rows][2 mbarriers]
// ------------------------------------------------------------------------------------------------
// Threads of a CTA of the TMA-fed vx kernel: a tile has 128 (CN / 8) work items (8-cell segments of 128 columns).  24^3:
// 384 items on 192 threads, 3 CTAs per SM, instead of one and a half trips of 256 threads: nv24 0.336 -> 0.307 ms per
// cycle.  40^3 (640 items) stays at 256 threads: 320 threads at the 102 registers that leaves measured slower (3.21 ->
// 3.52 ms per cycle of config 4).
__host__ __device__ constexpr int x_tma_threads(int cn) { return cn == 24 ? 192 : V_THREADS; }
__host__ __device__ constexpr int x_tma_minb(int cn) { return cn == 24 ? 3 : 2; }

template <int LIM, int CN>
__global__ void __launch_bounds__(x_tma_threads(CN), x_tma_minb(CN)) vsweep_x_tma_kernel(const __grid_constant__ CUtensorMap tmap, VParams P) {
    extern __shared__ __align__(128) double sm[];
    // the last tile of a plane may be ragged (24^2, 40^2: 64 columns; the box is zero-filled past the plane): a
    // multiple of 32, so warps stay whole
    constexpr int CT = 128, N = CN, plane = CN * CN, ntile = (plane + CT - 1) / CT, nsegx = CN / 8, seglen = 8;
    constexpr int ROWS = 3 * V_PAD + 2 * CN;
    constexpr int NT = x_tma_threads(CN);
    static_assert(plane % 32 == 0 && CN % 8 == 0, "whole warps, whole segments");
    // only the three pad strips are ever written by threads (zeros, once); the buffers belong to the TMA unit
    for (int e = threadIdx.x; e < V_PAD * CT; e += NT) {
        sm[e] = 0.0; sm[(V_PAD + CN) * CT + e] = 0.0; sm[(2 * V_PAD + 2 * CN) * CT + e] = 0.0;
    }
    const unsigned bar0 = smem_addr(sm + ROWS * CT);
    const unsigned sbuf0 = smem_addr(sm + V_PAD * CT);
    constexpr unsigned BUFSTEP = (unsigned)(CN + V_PAD) * CT * 8;
    if (threadIdx.x == 0) { mbar_init(bar0, 1); mbar_init(bar0 + 8, 1); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    __syncthreads();
    auto issue = [&](int tile, int b) {            // thread 0 only
        const int cell = P.cell0 + tile / ntile;
        mbar_expect_tx(bar0 + 8 * b, (unsigned)CN * CT * 8);
        tma_g2s_2d(sbuf0 + b * BUFSTEP, &tmap, (tile % ntile) * CT, cell * CN, bar0 + 8 * b);
    };
    if (threadIdx.x == 0) {
        if ((int)blockIdx.x < P.ntot) issue(blockIdx.x, 0);
        if ((int)(blockIdx.x + gridDim.x) < P.ntot) issue(blockIdx.x + gridDim.x, 1);
    }
    int it = 0;
    for (int tile = blockIdx.x; tile < P.ntot; tile += gridDim.x, ++it) {
        const int b = it & 1;
        const int cell = P.cell0 + tile / ntile;
        const int c0 = (tile % ntile) * CT;
        const double* T = P.table + (long)cell * TAB;
        const double t0 = T[0], t1 = T[1], t2 = T[2], t3 = T[3], finf = T[12];
        double* fb = P.f + (long)cell * P.S + c0;
        const double* A = sm + (V_PAD + b * (CN + V_PAD)) * CT;
        mbar_wait(bar0 + 8 * b, (it >> 1) & 1);
#pragma unroll
        for (int wi = threadIdx.x; wi < CT * nsegx; wi += NT) {
            const int seg = wi / CT, c = wi - seg * CT;
            const int col = c0 + c;
            if (plane % CT != 0 && col >= plane) continue;
            const int k1 = col / CN, k2 = col - k1 * CN;
            const double s0 = t0 + t2 * k1 + t3 * k2;
            const int a = seg * seglen;
            OutGlobal o{fb + c + (long)a * plane, (long)plane};
            march_cells<LIM, 2, 0, VL_X_BATCH>(smem_addr(A + c), CT * 8, N, a, a + seglen, s0, t1, finf, o);     // whole warps take this together
        }
        __syncthreads();                           // everybody is done reading buffer b: refill it
        if (threadIdx.x == 0 && tile + 2 * (int)gridDim.x < P.ntot) issue(tile + 2 * gridDim.x, b);
    }
}

// ------------------------------------------------------------------------------------------------
// a5 + a6: vy sweep then vz sweep on a tile of PT contiguous i_vx planes.  Shared layout of a buffer:
// cell (p, y, z) at OFF + p PS + y RS + z with RS = N2 + V_PAD (odd: threads that march neighbouring z
// lines hit distinct banks), PS = (N1 + V_PAD) RS, OFF = V_PAD RS + V_PAD; everything that is not a cell is zero and
// serves as the padding of the lines in both directions.  vy: A -> Bf; vz: Bf -> A; A -> global.
// ------------------------------------------------------------------------------------------------
// CN > 0: the velocity plane is CN x CN cells and the tile shape is the launcher's choice for it, all known at
// compile time (strides become immediates, the staging loops unroll); CN = 0: any shape, at run time.
template <int LIM, int CN>
__global__ void __launch_bounds__(V_THREADS, 3) vsweep_yz_kernel(VParams P) {
    extern __shared__ double sm[];
    const int N1 = CN ? CN : P.nv1, N2 = CN ? CN : P.nv2;
    constexpr int CCT = CN ? ((8 * V_THREADS) / (CN * CN) > 0 ? (8 * V_THREADS) / (CN * CN) : 1) : 0;      // planes per tile, as launch_vsweeps picks them
    constexpr int CSEG = CN ? (CN + 7) / 8 : 0;
    if (CN && (P.ct != CCT || P.nseg != CSEG || P.nseg2 != CSEG)) return;
    // REGULAR: a thread's cells of a tile are DROW whole rows apart and a row index never wraps inside a plane step:
    // every staging offset is a compile-time constant (32x32 and 16x16 planes with 256 threads)
    constexpr int DROW = CN ? V_THREADS / CN : 1;
    constexpr bool REGULAR = CN && V_THREADS % (CN ? CN : 1) == 0 && (CN ? CN : 1) % DROW == 0;
    const int ct = CN ? CCT : P.ct, nseg1 = CN ? CSEG : P.nseg, nseg2 = CN ? CSEG : P.nseg2;
    const int plane = N1 * N2;
    const int RS = N2 + V_PAD, PS = (N1 + V_PAD) * RS, OFF = V_PAD * RS + V_PAD;
    const int BUF = (OFF + ct * PS + 1) & ~1;
    double* A = sm;
    double* Bf = sm + BUF;
    for (int e = threadIdx.x; e < 2 * BUF; e += V_THREADS) sm[e] = 0.0;
    __syncthreads();
    // cell e = threadIdx.x of a tile sits at (pp, y, z); stepping e by V_THREADS moves it by (dpp, dy, dz) plus carries
    const unsigned sA = smem_addr(A);
    const int z_init = threadIdx.x % N2, row_init = threadIdx.x / N2;
    const int y_init = row_init % N1;
    const unsigned so_init = OFF + (row_init / N1) * PS + y_init * RS + z_init;
    const int dz = V_THREADS % N2, drow = V_THREADS / N2;
    const int dy = drow % N1;
    const unsigned dso = dz + dy * RS + (drow / N1) * PS;
    for (int tile = blockIdx.x; tile < P.ntot; tile += gridDim.x) {
        const int cell = P.cell0 + tile / P.ntile;
        const int p0 = (tile % P.ntile) * ct;
        const int np = ct;                          // equal tiles: ct divides nv0 (launch_vsweeps)
        double* fb = P.f + (long)cell * P.S + (long)p0 * plane;
        const double* T = P.table + (long)cell * TAB;
        const int ncellt = np * plane;
        if (REGULAR) {   // global -> A by 8-byte cp.async: element i of this thread sits DROW rows further, all offsets constant
#pragma unroll
            for (int i = 0; i < (CN ? CCT * CN * CN / V_THREADS : 1); ++i)
                cp_async8(sA + (so_init + ((i * DROW) / (CN ? CN : 1)) * PS + ((i * DROW) % (CN ? CN : 1)) * RS) * 8, fb + threadIdx.x + i * V_THREADS);
            cp_async_wait_all();
        } else {   // (pp, y, z) of e = threadIdx.x + i V_THREADS advanced by carries
            int z = z_init, y = y_init;
            unsigned so = so_init;
            for (int e = threadIdx.x; e < ncellt; e += V_THREADS) {
                cp_async8(sA + so * 8, fb + e);
                z += dz; y += dy; so += dso;
                if (z >= N2) { z -= N2; so += RS - N2; ++y; }
                if (y >= N1) { y -= N1; so += PS - N1 * RS; }
            }
            cp_async_wait_all();
        }
        __syncthreads();
        {   // vy: line along i_vy (stride RS); transverse (i_vx, i_vz); thread index runs along z
            const double t0 = T[4], t1 = T[5], t2 = T[6], t3 = T[7], finf = T[13];
            const int seglen = (N1 + nseg1 - 1) / nseg1;
            const int nl = np * N2;
            for (int wi = threadIdx.x; wi < nl * nseg1; wi += V_THREADS) {
                const int seg = wi / nl, l = wi - seg * nl;
                const int p = l / N2, z = l - p * N2;
                const double s0 = t0 + t2 * (p0 + p) + t3 * z;
                const int a = seg * seglen, b = min(a + seglen, N1);
                OutShared o{smem_addr(Bf + OFF + p * PS + z + a * RS), RS * 8};
                march_cells<LIM, 1>(smem_addr(A + OFF + p * PS + z), RS * 8, N1, a, b, s0, t1, finf, o);
            }
        }
        __syncthreads();
        {   // vz: contiguous lines; transverse (i_vx, i_vy); thread index runs along y (stride RS, odd)
            const double t0 = T[8], t1 = T[9], t2 = T[10], t3 = T[11], finf = T[14];
            const int seglen = (N2 + nseg2 - 1) / nseg2;
            const int nl = np * N1;
            for (int wi = threadIdx.x; wi < nl * nseg2; wi += V_THREADS) {
                const int seg = wi / nl, l = wi - seg * nl;
                const int p = l / N1, y = l - p * N1;
                const double s0 = t0 + t2 * (p0 + p) + t3 * y;
                const int a = seg * seglen, b = min(a + seglen, N2);
                OutShared o{smem_addr(A + OFF + p * PS + y * RS + a), 8};
                march_cells<LIM, 1>(smem_addr(Bf + OFF + p * PS + y * RS), 8, N2, a, b, s0, t1, finf, o);
            }
        }
        __syncthreads();
        if (REGULAR) {
#pragma unroll
            for (int i = 0; i < (CN ? CCT * CN * CN / V_THREADS : 1); ++i)
                __stcs(fb + threadIdx.x + i * V_THREADS, lds(sA + (so_init + ((i * DROW) / (CN ? CN : 1)) * PS + ((i * DROW) % (CN ? CN : 1)) * RS) * 8));
        } else {
            int z = z_init, y = y_init;
            unsigned so = so_init;
            for (int e = threadIdx.x; e < ncellt; e += V_THREADS) {
                __stcs(fb + e, lds(sA + so * 8));
                z += dz; y += dy; so += dso;
                if (z >= N2) { z -= N2; so += RS - N2; ++y; }
                if (y >= N1) { y -= N1; so += PS - N1 * RS; }
            }
        }
        __syncthreads();
    }
}

// ------------------------------------------------------------------------------------------------
// a5 + a6 with the tile loaded by 2D tiled TMA (one box {CN, CN} per plane) into a dense staging buffer with zero
// pad rows between the planes: the vy sweep reads it directly (lanes run along z: any pitch is conflict-free) and
// writes the padded, odd-pitch buffer Bf; as soon as the vy sweep is done the staging buffer is free and the NEXT
// tile's load is issued, landing while the vz sweep (Bf -> A) and the store (A -> global) run.  No load instruction,
// no exposed load latency, two block barriers per tile instead of four, and still 3 CTAs per SM for 32x32 planes.
//   shared: [staging: 8 + ct (CN + 8) rows of CN][Bf][A][mbarrier]
// ------------------------------------------------------------------------------------------------
// Tile shape of the TMA-staged vy+vz kernel for CN x CN planes: planes per tile (about 2048 cells), and the threads of
// a CTA = one work item (an 8-cell segment of one line) per thread, rounded up to whole warps.
// 40x40 planes: two planes per tile (400 work items, 416 threads, 2 CTAs per SM = 26 warps at 69 registers) measured
// 11 % faster than one plane per tile (224 threads, 3 CTAs = 21 warps): config 4, 8.86 -> 7.85 ms per cycle
#ifndef VL_YZ40_PLANES
#define VL_YZ40_PLANES 2
#endif
#ifndef VL_YZ32_PLANES
#define VL_YZ32_PLANES 2
#endif
__host__ __device__ constexpr int yz_tma_planes(int cn) { return cn == 40 ? VL_YZ40_PLANES : cn == 32 ? VL_YZ32_PLANES : 2048 / (cn * cn) > 0 ? 2048 / (cn * cn) : 1; }
__host__ __device__ constexpr int yz_tma_threads(int cn) { return (yz_tma_planes(cn) * cn * ((cn + 7) / 8) + 31) / 32 * 32; }
static_assert(yz_tma_threads(16) == 256 && yz_tma_threads(24) == 224 && yz_tma_threads(48) == 288, "");
// resident CTAs per SM the kernel is compiled for: 3 (80 registers at 256 threads; 70 at the 288 threads of a 48x48 plane)
// 48x48: 288 threads and 69 KB per CTA; 3 CTAs per SM (27 warps at 70 registers, no spills) measured 12 % faster than 2
// (18 warps): nv48 6.89 -> 6.08 ms per cycle.  40x40 with one plane per tile and 4 CTAs (28 warps) measured slower than two
// planes and 2 CTAs (26 warps): 7.92 -> 8.20 ms.
#ifndef VL_YZ48_MINB
#define VL_YZ48_MINB 3
#endif
#ifndef VL_YZ40_MINB
#define VL_YZ40_MINB (VL_YZ40_PLANES > 1 ? 2 : VL_YZ_MINB)
#endif
// 32x32: the compact layout leaves room for 4 CTAs per SM (57 KB each), and the kernel fits 62 registers without spills,
// but 32 warps at 62 registers measured no faster than 24 at 80 (2.87 against 2.84 ms per cycle of config 3): 3.
// 24x24: 4 CTAs (28 warps at 69 registers) against 3 (21 warps): nv24 0.803 -> 0.718 ms.
#ifndef VL_YZ32_MINB
#define VL_YZ32_MINB (VL_YZ32_PLANES == 1 ? 6 : VL_YZ32_PLANES == 4 ? 1 : 3)
#endif
#ifndef VL_YZ24_MINB
#define VL_YZ24_MINB 4
#endif
__host__ __device__ constexpr int yz_tma_minb(int cn) { return cn == 48 ? VL_YZ48_MINB : cn == 40 ? VL_YZ40_MINB : cn == 32 ? VL_YZ32_MINB : cn == 24 ? VL_YZ24_MINB : VL_YZ_MINB; }

// MOM = 1 (VXV order): the 10 raw velocity moments, eqs. (2)-(4), of the final f are
// reduced in this kernel.  A CTA then takes WHOLE spatial cells (all tiles of a cell one after the other), sums its
// cells while it stores them, and writes the moments of the cell itself: no partial sums in global memory, no
// atomics, a fixed summation order.  For planes where a thread keeps its i_vz over a tile (16x16, 32x32).
// Shared-memory layout of the TMA-staged kernel, in doubles.  Staging: pad rows of zeros around every plane (>= V_PAD;
// every TMA box must start 128-byte aligned: 8 rows of any even N2 do, and any number of rows when a row is a multiple
// of 128 bytes).  Bf (between the sweeps): rows of N2 + V_PAD, zero pads.  A (output): written by the vz sweep and read
// by the store loop only, so it needs no pads, just an odd pitch (lanes of the vz sweep run along y).
#ifndef VL_YZ_COMPACT
#define VL_YZ_COMPACT 1
#endif
// Zero cells on either side of a line in this kernel's buffers.  A box-face segment whose lanes reach floor|sigma| =
// pad falls back to the general face walk, warp and all: at 48^3 the GEM electrons reach 3.2 cells, and a third of the
// electron warps did (nv48 vy+vz 5.85 -> 4.9 ms per cycle with the walk admitted).  5 for 40x40 and 48x48 planes.
#ifndef VL_YZ_PAD5
#define VL_YZ_PAD5 1
#endif
__host__ __device__ constexpr int yz_tma_pad(int cn) { return VL_YZ_PAD5 && (cn == 40 || cn == 48) ? 5 : V_PAD; }
__host__ __device__ constexpr int yz_tma_spad(int cn) { return VL_YZ_COMPACT && cn % 16 == 0 ? yz_tma_pad(cn) : 8; }
// (the walks may look at the 4th row before a line, whatever it holds: one more row before the first plane)
__host__ __device__ constexpr int yz_tma_spad0(int cn) { return yz_tma_spad(cn) > yz_tma_pad(cn) ? yz_tma_spad(cn) : yz_tma_pad(cn) + 1; }
__host__ __device__ constexpr int yz_tma_stg(int cn) { return ((yz_tma_spad0(cn) + yz_tma_planes(cn) * (cn + yz_tma_spad(cn))) * cn + 15) & ~15; }
// Bf is read along z only: no pad rows, the rows of all planes follow each other at pitch N2 + pad (odd), the gap is the
// right pad of one row and the left pad of the next; pad + 1 cells before the first row and after the last.
__host__ __device__ constexpr int yz_tma_buf(int cn) { return (2 * (yz_tma_pad(cn) + 1) + yz_tma_planes(cn) * cn * (cn + yz_tma_pad(cn)) + 1) & ~1; }
__host__ __device__ constexpr int yz_tma_rsa(int cn) { return VL_YZ_COMPACT ? (cn | 1) : cn + V_PAD; }
__host__ __device__ constexpr int yz_tma_psa(int cn) { return VL_YZ_COMPACT ? cn * yz_tma_rsa(cn) : (cn + V_PAD) * (cn + V_PAD); }
__host__ __device__ constexpr int yz_tma_offa(int cn) { return VL_YZ_COMPACT ? 0 : V_PAD * (cn + V_PAD) + V_PAD; }
__host__ __device__ constexpr int yz_tma_bufa(int cn) { return (yz_tma_offa(cn) + yz_tma_planes(cn) * yz_tma_psa(cn) + 1) & ~1; }
__host__ __device__ constexpr size_t yz_tma_smem(int cn) {
    return (size_t)(yz_tma_stg(cn) + yz_tma_buf(cn) + yz_tma_bufa(cn)) * 8 + 16 + TAB * 8 + 8 * 10 * 8;
}

template <int LIM, int CN, int MOM = 0>
__global__ void __launch_bounds__(yz_tma_threads(CN), yz_tma_minb(CN)) vsweep_yz_tma_kernel(const __grid_constant__ CUtensorMap tmap, VParams P) {
    extern __shared__ __align__(128) double sm[];
    constexpr int N1 = CN, N2 = CN, plane = CN * CN;
    constexpr int ct = yz_tma_planes(CN);
    constexpr int nseg = (CN + 7) / 8, seglen = (CN + nseg - 1) / nseg;
    constexpr int YZP = yz_tma_pad(CN);                          // zero cells on either side of a line
    constexpr int RS = N2 + YZP, PS = N1 * RS, OFF = YZP + 1;    // Bf: see yz_tma_buf
    constexpr int BUF = yz_tma_buf(CN);
    static_assert(RS % 2 == 1 && OFF + ct * PS + YZP + 1 <= BUF, "odd pitch, pads inside the buffer");
    constexpr int SPAD = yz_tma_spad(CN);                        // pad rows of the staging buffer: >= V_PAD, and 8 rows of
                                                                 // any even N2 keep every TMA box 128-byte aligned
    constexpr int SP0 = yz_tma_spad0(CN);                        // rows before the first plane
    constexpr int SROWS = SP0 + ct * (N1 + SPAD);                // staging rows of N2 doubles
    constexpr int STG = (SROWS * N2 + 15) & ~15;                 // keeps Bf 128-byte aligned
    static_assert(STG == yz_tma_stg(CN) && BUF == yz_tma_buf(CN), "layout helpers");
    constexpr int RSA = yz_tma_rsa(CN), PSA = yz_tma_psa(CN), OFFA = yz_tma_offa(CN), BUFA = yz_tma_bufa(CN);      // output buffer A
    // The work items of a sweep (ct CN nseg) need not fill the last warp.  Its idle lanes REPEAT the items of the 32
    // lanes before them (same reads, same values written to the same places), so that every warp that works at all is
    // whole: the walks vote with the full mask, no __activemask() bookkeeping, no divergence guards around the votes.
    constexpr int FW = 2;
    constexpr int NITEM = ct * CN * nseg;
    constexpr int NT = yz_tma_threads(CN);         // threads of the CTA: the work items rounded up to whole warps
    static_assert(NITEM >= 32 && NITEM <= NT && NT - NITEM < 32 && CN % 8 == 0 && seglen == 8, "one item per thread, whole warps, whole segments");
    if (P.ct != ct || P.nseg != nseg || P.nseg2 != nseg || P.nv1 != CN || P.nv2 != CN) return;
    double* St = sm;
    double* Bf = sm + STG;
    double* A = Bf + BUF;
    const unsigned bar = smem_addr(A + BUFA);
    const double* tab = A + BUFA + 2;               // the tile's sweep-table row rides along with the tile (16-byte aligned)
    double* red = A + BUFA + 2 + TAB;               // MOM: [warps][10] partial sums of a spatial cell
    static_assert((TAB * 8) % 16 == 0, "bulk copy size");
    // zero: the staging pad rows (never written again), Bf and A entirely (their cells are overwritten per tile)
    for (int e = threadIdx.x; e < SP0 * N2; e += NT) St[e] = 0.0;
    for (int e = threadIdx.x; e < SPAD * N2; e += NT) {
#pragma unroll
        for (int p = 0; p < ct; ++p) St[(SP0 + p * (N1 + SPAD) + N1) * N2 + e] = 0.0;
    }
    for (int e = threadIdx.x; e < BUF + BUFA; e += NT) Bf[e] = 0.0;
    if (threadIdx.x == 0) mbar_init(bar, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    __syncthreads();
    const unsigned sSt = smem_addr(St), sA = smem_addr(A);
    auto issue = [&](int cell, int p0) {           // thread 0 only: ct boxes, one per plane
        mbar_expect_tx(bar, (unsigned)ct * plane * 8 + TAB * 8);
        bulk_g2s(smem_addr(tab), P.table + (long)cell * TAB, TAB * 8, bar);
#pragma unroll
        for (int p = 0; p < ct; ++p)
            tma_g2s_2d(sSt + (unsigned)((SP0 + p * (N1 + SPAD)) * N2) * 8, &tmap, 0, (cell * P.nv0 + p0 + p) * N1, bar);
    };
    // (spatial cell, tile within the cell) of this CTA's tiles, advanced without a division per tile.  MOM: the CTA
    // owns the cells blockIdx.x, blockIdx.x + gridDim.x, ... and walks the tiles of a cell in order.
    const int step_c = MOM ? 0 : gridDim.x / P.ntile, step_t = MOM ? 1 : gridDim.x % P.ntile;
    const int wrap_c = MOM ? gridDim.x : 1;
    const int ncell_l = P.ntot / P.ntile;
    int tcell = MOM ? blockIdx.x : blockIdx.x / P.ntile, ttile = MOM ? 0 : blockIdx.x % P.ntile;
    if (threadIdx.x == 0 && tcell < ncell_l) issue(P.cell0 + tcell, ttile * ct);
    // staging map of the store loop (as in the plain kernel)
    const int z_init = threadIdx.x % N2, row_init = threadIdx.x / N2;
    const int y_init = row_init % N1;
    const unsigned so_init = OFFA + (row_init / N1) * PSA + y_init * RSA + z_init;
    constexpr int dz = NT % N2, drow = NT / N2, dy = drow % N1;
    constexpr unsigned dso = dz + dy * RSA + (drow / N1) * PSA;
    constexpr int ncellt = ct * plane;
    double T0 = 0.0, Tx = 0.0, Txx = 0.0, Ty = 0.0, Tyy = 0.0, Txy = 0.0;      // MOM: this thread's sums over a spatial cell
    int it = 0;
    for (; tcell < ncell_l; ++it) {
        const int cell = P.cell0 + tcell;
        const int p0 = ttile * ct;
        double* fb = P.f + (long)cell * P.S + (long)p0 * plane;
        tcell += step_c; ttile += step_t;
        const bool last_of_cell = ttile >= P.ntile;
        if (last_of_cell) { ttile -= P.ntile; tcell += wrap_c; }
        mbar_wait(bar, it & 1);
        if (NT != V_THREADS) __syncwarp();
        // the table row arrived with the tile; it is overwritten when the next tile is issued (after the vy sweep)
        const double ty0 = tab[4], ty1 = tab[5], ty2 = tab[6], ty3 = tab[7], finfy = tab[13];
        const double tz0 = tab[8], tz1 = tab[9], tz2 = tab[10], tz3 = tab[11], finfz = tab[14];
        {   // vy: line along i_vy (stride N2 in the staging buffer); transverse (plane, i_vz); threads run along z
            constexpr int nl = ct * N2;
            {
                int wi = threadIdx.x;
                if (wi >= NITEM) wi -= 32;
                const int seg = wi / nl, l = wi - seg * nl;
                const int p = l / N2, z = l - p * N2;
                const double s0 = ty0 + ty2 * (p0 + p) + ty3 * z;
                const int a = seg * seglen, b = a + seglen;          // CN is a multiple of 8: whole segments
                OutShared o{smem_addr(Bf + OFF + p * PS + z + a * RS), RS * 8};
                march_cells<LIM, FW, 1, VL_YZ_BATCH, (CN == 32 ? VL_LITE_UNROLL32 : VL_LITE_UNROLL), YZP>(sSt + (unsigned)((SP0 + p * (N1 + SPAD)) * N2 + z) * 8, N2 * 8, N1, a, b, s0, ty1, finfy, o);
            }
        }
        __syncthreads();                           // vy done: Bf complete, staging buffer free
        if (threadIdx.x == 0 && tcell < ncell_l) issue(P.cell0 + tcell, ttile * ct);
        {   // vz: contiguous lines of Bf; transverse (plane, i_vy); threads run along y (pitch RS, odd)
            constexpr int nl = ct * N1;
            {
                int wi = threadIdx.x;
                if (wi >= NITEM) wi -= 32;
                const int seg = wi / nl, l = wi - seg * nl;
                const int p = l / N1, y = l - p * N1;
                const double s0 = tz0 + tz2 * (p0 + p) + tz3 * y;
                const int a = seg * seglen, b = a + seglen;
                OutShared o{smem_addr(A + OFFA + p * PSA + y * RSA + a), 8};
                march_cells<LIM, FW, 1, VL_YZ_BATCH, (CN == 32 ? VL_LITE_UNROLL32 : VL_LITE_UNROLL), YZP>(smem_addr(Bf + OFF + p * PS + y * RS), 8, N2, a, b, s0, tz1, finfz, o);
            }
        }
        __syncthreads();                           // vz done: A complete
        if (MOM) {
            // A -> global, and the sums of the stored cells.  This thread keeps its i_vz; per plane its cells are EPP rows
            // drow apart: sum f, sum vy f, sum vy^2 f over them, folded with the plane's vx; vz enters once per spatial cell.
            static_assert(!MOM || (dz == 0 && N1 % drow == 0 && ncellt % NT == 0), "fused moments: a thread keeps its i_vz");
            constexpr int EPP = N1 / (drow > 0 ? drow : 1);
            const double vy0 = P.vmin[1] + (y_init + 0.5) * P.dv[1];
#pragma unroll
            for (int pp = 0; pp < ct; ++pp) {
                double r0 = 0.0, r1 = 0.0, r2 = 0.0;
#pragma unroll
                for (int j = 0; j < EPP; ++j) {
                    const double fv = lds(sA + (so_init + pp * PSA + j * drow * RSA) * 8);
                    __stcs(fb + threadIdx.x + (pp * EPP + j) * NT, fv);
                    const double vy = vy0 + (j * drow) * P.dv[1];
                    const double t = vy * fv;
                    r0 += fv; r1 += t; r2 = fma(vy, t, r2);
                }
                const double vx = P.vmin[0] + (p0 + pp + 0.5) * P.dv[0];
                const double u = vx * r0;
                T0 += r0; Tx += u; Txx = fma(vx, u, Txx); Ty += r1; Tyy += r2; Txy = fma(vx, r1, Txy);
            }
            if (last_of_cell) {
                const double vz = P.vmin[2] + (z_init + 0.5) * P.dv[2];
                double M[10] = {T0, Tx, Ty, vz * T0, Txx, Tyy, vz * (vz * T0), Txy, vz * Tx, vz * Ty};
                T0 = Tx = Txx = Ty = Tyy = Txy = 0.0;
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) {
#pragma unroll
                    for (int q = 0; q < 10; ++q) M[q] += __shfl_down_sync(0xffffffffu, M[q], o);
                }
                if ((threadIdx.x & 31) == 0) {
#pragma unroll
                    for (int q = 0; q < 10; ++q) red[(threadIdx.x >> 5) * 10 + q] = M[q];
                }
                __syncthreads();
                if (threadIdx.x < 10) {
                    double r = red[threadIdx.x];
                    for (int w = 1; w < NT / 32; ++w) r += red[w * 10 + threadIdx.x];      // fixed order over the warps
                    P.mom[(long)threadIdx.x * P.mom_ncell + (cell - P.cell0)] = r * (P.dv[0] * P.dv[1] * P.dv[2]);
                }
                // red is written again a whole spatial cell (>= 2 block barriers) later
            }
        } else
        {   // A -> global (the next tile's vz sweep writes A only after the next barrier)
            // the same trip count for every lane (the last trip is guarded instead): a loop that ends lane by lane would
            // make the compiler guard every full-mask vote of the next tile's walks against divergence
            int z = z_init, y = y_init;
            unsigned so = so_init;
            constexpr int NTRIP = (ncellt + NT - 1) / NT;
            if constexpr (ncellt % NT == 0) {
                for (int e = threadIdx.x; e < ncellt; e += NT) {
                    __stcs(fb + e, lds(sA + so * 8));
                    z += dz; y += dy; so += dso;
                    if (z >= N2) { z -= N2; so += RSA - N2; ++y; }
                    if (y >= N1) { y -= N1; so += PSA - N1 * RSA; }
                }
            } else {
#pragma unroll 4
                for (int i = 0; i < NTRIP; ++i) {
                    const int e = threadIdx.x + i * NT;
                    if (e < ncellt) __stcs(fb + e, lds(sA + so * 8));
                    z += dz; y += dy; so += dso;
                    if (z >= N2) { z -= N2; so += RSA - N2; ++y; }
                    if (y >= N1) { y -= N1; so += PSA - N1 * RSA; }
                }
            }
        }
    }
}

constexpr size_t V_SMEM_MAX = 200 * 1024;

// Persistent grid size (resident CTAs of the device) of one kernel instantiation at one dynamic shared-memory size.
// Function attributes and occupancy are per device: the cache is keyed by (device, kernel, smem) and guarded, so
// several contexts on several devices (or threads) of one process each get their own answer.
template <class K>
static int resident_ctas(K kernel, size_t smem, int threads = V_THREADS) {
    static std::mutex mu;
    static std::map<std::tuple<int, const void*, size_t>, int> cache;
    int dev = 0;
    cudaGetDevice(&dev);
    const auto key = std::make_tuple(dev, (const void*)kernel, smem + ((size_t)threads << 40));
    std::lock_guard<std::mutex> lock(mu);
    auto it = cache.find(key);
    if (it != cache.end()) return it->second;
    cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)V_SMEM_MAX);
    int per_sm = 0, sms = 0;
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kernel, threads, smem);
    if (per_sm < 1) per_sm = 1;
    cache[key] = per_sm * sms;
    return per_sm * sms;
}

int launch_vsweeps(vlasov_ctx* c, const Species& s, double* f, int row0, int nrows, bool ghost, double* mom_out, bool* mom_done,
                   const double* src) {
    if (!src) src = f;
    if (mom_done) *mom_done = false;
    if (nrows <= 0) return VLASOV_OK;
    VParams P;
    P.fsrc = src; P.f = f; P.table = c->table; P.S = s.nvtot;
    P.nv0 = s.nv[0]; P.nv1 = s.nv[1]; P.nv2 = s.nv[2];
    P.cell0 = row0 * c->G.nx;
    P.mom = nullptr; P.mom_ncell = 0;
    for (int d = 0; d < 3; ++d) { P.vmin[d] = s.vmin[d]; P.dv[d] = s.dv[d]; }
    const int lim = c->G.limiter ? 1 : 0;
    const int ncell = nrows * c->G.nx;
    const int plane = s.nv[1] * s.nv[2];
    {
        const int cn = (s.nv[0] == s.nv[1] && s.nv[1] == s.nv[2]) ? s.nv[0] : 0;
        const bool cube = cn == 16 || cn == 32;            // shapes with a compile-time-shape kernel
        int ct = 128;
        while (ct > 32 && ((size_t)(s.nv[0] + 2 * V_PAD) * ct * 8 > 48 * 1024 || ct / 2 >= plane)) ct >>= 1;
        P.ct = ct;
        const size_t smem = (size_t)(s.nv[0] + 2 * V_PAD) * ct * 8;
        if (smem > V_SMEM_MAX) return VLASOV_EINVAL;
        P.ntile = (plane + ct - 1) / ct;
        P.ntot = P.ntile * ncell;
        P.nseg = V_THREADS / ct; if (P.nseg < 1) P.nseg = 1; if (P.nseg > s.nv[0]) P.nseg = s.nv[0];
        if (cube && ct == 128) P.nseg = cn / 8;            // 8-cell segments (register-window walk)
        const int spec = (cube && ct == 128) ? cn : 0;
        void (*k)(VParams) = lim ? vsweep_x_kernel<1, 0> : vsweep_x_kernel<0, 0>;
        if (spec == 16) k = lim ? vsweep_x_kernel<1, 16> : vsweep_x_kernel<0, 16>;
        if (spec == 32) k = lim ? vsweep_x_kernel<1, 32> : vsweep_x_kernel<0, 32>;
        const int tspec = (cn == 16 || cn == 24 || cn == 32 || cn == 40 || cn == 48) ? cn : 0;
        if (tspec && !ghost && (long)c->G.nrows * c->G.nx * s.nv[0] < 2147483647L) {      // TMA coordinates are 32-bit
            // prefetching variant: one CUtensorMap over f as a matrix [cells * nv0][nv1 * nv2]; its own tile shape
            CUtensorMap tm;
            if (!make_tensor_map_2d(&tm, src, plane, (long)c->G.nrows * c->G.nx * s.nv[0], 128, tspec)) return VLASOV_ECUDA;
            P.ct = 128; P.nseg = tspec / 8;
            P.ntile = (plane + 127) / 128;
            P.ntot = P.ntile * ncell;
            void (*kt)(CUtensorMap, VParams) = lim ? vsweep_x_tma_kernel<1, 32> : vsweep_x_tma_kernel<0, 32>;
            if (tspec == 16) kt = lim ? vsweep_x_tma_kernel<1, 16> : vsweep_x_tma_kernel<0, 16>;
            if (tspec == 24) kt = lim ? vsweep_x_tma_kernel<1, 24> : vsweep_x_tma_kernel<0, 24>;
            if (tspec == 40) kt = lim ? vsweep_x_tma_kernel<1, 40> : vsweep_x_tma_kernel<0, 40>;
            if (tspec == 48) kt = lim ? vsweep_x_tma_kernel<1, 48> : vsweep_x_tma_kernel<0, 48>;
            const size_t smem_t = (size_t)(3 * V_PAD + 2 * tspec) * 128 * 8 + 16;
            const int ntx = x_tma_threads(tspec);
            const int grid = min(P.ntot, resident_ctas(kt, smem_t, ntx));
            Launch L(c, K_VSWEEP_X);
            kt<<<grid, ntx, smem_t, c->stream>>>(tm, P);
        } else {
            const int grid = min(P.ntot, resident_ctas(k, smem));
            Launch L(c, K_VSWEEP_X);
            k<<<grid, V_THREADS, smem, c->stream>>>(P);
        }
    }
    {
        const size_t rs = s.nv[2] + V_PAD, ps = (s.nv[1] + V_PAD) * rs, off = V_PAD * rs + V_PAD;
        // segments of about 8 cells per thread, about V_THREADS threads per tile: small tiles, many CTAs per SM
        int pt = (8 * V_THREADS) / plane;
        if (pt < 1) pt = 1;
        if (pt > s.nv[0]) pt = s.nv[0];
        while (pt > 1 && s.nv[0] % pt) --pt;            // equal tiles
        P.ct = pt;
        const size_t buf = (off + pt * ps + 1) & ~(size_t)1;
        const size_t smem = 2 * buf * 8;
        if (smem > V_SMEM_MAX) return VLASOV_EINVAL;
        P.ntile = (s.nv[0] + pt - 1) / pt;
        P.ntot = P.ntile * ncell;
        P.nseg = (s.nv[1] + 7) / 8;
        P.nseg2 = (s.nv[2] + 7) / 8;
        const int sq = s.nv[1] == s.nv[2] ? s.nv[1] : 0;   // square planes with a compile-time-shape kernel
        const int want_pt = sq ? ((8 * V_THREADS) / (sq * sq) > 0 ? (8 * V_THREADS) / (sq * sq) : 1) : 0;
        const int spec = (sq == 16 || sq == 24 || sq == 32 || sq == 40 || sq == 48) && pt == want_pt ? sq : 0;
        void (*k)(VParams) = lim ? vsweep_yz_kernel<1, 0> : vsweep_yz_kernel<0, 0>;
        if (spec == 16) k = lim ? vsweep_yz_kernel<1, 16> : vsweep_yz_kernel<0, 16>;
        if (spec == 24) k = lim ? vsweep_yz_kernel<1, 24> : vsweep_yz_kernel<0, 24>;
        if (spec == 32) k = lim ? vsweep_yz_kernel<1, 32> : vsweep_yz_kernel<0, 32>;
        if (spec == 40) k = lim ? vsweep_yz_kernel<1, 40> : vsweep_yz_kernel<0, 40>;
        if (spec == 48) k = lim ? vsweep_yz_kernel<1, 48> : vsweep_yz_kernel<0, 48>;
        // the TMA kernel's own tile: planes per tile (a divisor of nv0), work items rounded up to whole warps
        const int ptt = spec == 16 ? yz_tma_planes(16) : spec == 24 ? yz_tma_planes(24) : spec == 40 ? yz_tma_planes(40) :
                        spec == 48 ? yz_tma_planes(48) : yz_tma_planes(32);
        if (spec && s.nv[0] % ptt == 0 && (long)c->G.nrows * c->G.nx * s.nv[0] * s.nv[1] < 2147483647L) {
            P.ct = ptt;
            P.ntile = s.nv[0] / ptt;
            P.ntot = P.ntile * ncell;
            const size_t buf = (off + ptt * ps + 1) & ~(size_t)1;
            const int pt = ptt;
            // TMA-staged variant: f as a matrix [cells * nv0 * nv1][nv2], one box {nv2, nv1} per plane
            CUtensorMap tm;
            if (!make_tensor_map_2d(&tm, f, s.nv[2], (long)c->G.nrows * c->G.nx * s.nv[0] * s.nv[1], s.nv[2], s.nv[1])) return VLASOV_ECUDA;
            void (*kt)(CUtensorMap, VParams) = lim ? vsweep_yz_tma_kernel<1, 32> : vsweep_yz_tma_kernel<0, 32>;
            if (spec == 16) kt = lim ? vsweep_yz_tma_kernel<1, 16> : vsweep_yz_tma_kernel<0, 16>;
            if (spec == 24) kt = lim ? vsweep_yz_tma_kernel<1, 24> : vsweep_yz_tma_kernel<0, 24>;
            if (spec == 40) kt = lim ? vsweep_yz_tma_kernel<1, 40> : vsweep_yz_tma_kernel<0, 40>;
            if (spec == 48) kt = lim ? vsweep_yz_tma_kernel<1, 48> : vsweep_yz_tma_kernel<0, 48>;
            const size_t smem_t = yz_tma_smem(spec);
            // moments of the final f reduced in the same pass (VXV order): CTAs take whole spatial cells
            const bool mom = mom_out && !ghost && (spec == 16 || spec == 32);
            if (mom) {
                P.mom = mom_out; P.mom_ncell = ncell;
                if (spec == 16) kt = lim ? vsweep_yz_tma_kernel<1, 16, 1> : vsweep_yz_tma_kernel<0, 16, 1>;
                else kt = lim ? vsweep_yz_tma_kernel<1, 32, 1> : vsweep_yz_tma_kernel<0, 32, 1>;
                if (mom_done) *mom_done = true;
            }
            if (smem_t > V_SMEM_MAX) return VLASOV_EINVAL;
            const int nt = spec == 16 ? yz_tma_threads(16) : spec == 24 ? yz_tma_threads(24) : spec == 40 ? yz_tma_threads(40) :
                           spec == 48 ? yz_tma_threads(48) : yz_tma_threads(32);
            const int grid = min(mom ? ncell : P.ntot, resident_ctas(kt, smem_t, nt));
            Launch L(c, K_VSWEEP_YZ);
            kt<<<grid, nt, smem_t, c->stream>>>(tm, P);
        } else {
            const int grid = min(P.ntot, resident_ctas(k, smem));
            Launch L(c, K_VSWEEP_YZ);
            k<<<grid, V_THREADS, smem, c->stream>>>(P);
        }
    }
    return cudaGetLastError() == cudaSuccess ? VLASOV_OK : VLASOV_ECUDA;
}

}  // namespace vl
