// Internal declarations of libvlasov_b200 (CUDA path).  Shares nothing with oracle/.
// Citations: PAPER.md:<line> + equation; readings R* are in DESIGN.md.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include "../../include/vlasov.h"

namespace vl {

constexpr int MAX_SPECIES = 8;
// per-spatial-cell sweep table, 16 doubles per cell:
//   [4*d + 0..3], d = 0,1,2: sigma(k, k1, k2) = c0 + c1*k + c2*k1 + c3*k2 for face k (between cells
//   k-1 and k) of the line with transverse cell indices (k1, k2) -- d=0: (ivy, ivz); d=1: (ivx, ivz);
//   d=2: (ivx, ivy).  [12 + d]: f_infinity of sweep d.  [15]: multiplicative scale applied to the
//   source block before the first sweep (ghost fill), 1 otherwise.  [16]: spatial cell the first sweep
//   READS (ghost fill: the edge cell, R15a; otherwise the cell itself), stored as a double.
constexpr int TAB = 20;

struct Species {
    double q, m;
    int nv[3];
    double vmin[3], dv[3];
    double f_inf;
    long nvtot;        // nv[0]*nv[1]*nv[2]
    double* f;         // caller's buffer
    const double* fluid[2];   // fluid5 of y_lo / y_hi (device), or null
};

struct Geom {
    int nx, ny, g, nyg;
    int nz, nrows;     // 3D3V: slabs along z (1 = the 2D path); nrows = nz * nyg = all rows of an array
    double dx, dy, dz;
    int bc_lo, bc_hi;
    int limiter, fields_yee, wall;
};

}  // namespace vl

struct vlasov_ctx {
    vl::Geom G;
    int order;
    double c, mu0;
    int ns;
    vl::Species sp[vl::MAX_SPECIES];
    cudaStream_t stream;
    // scratch carve-up (device)
    double* pong;        // ping-pong copy of one species' f
    double* table;       // [nyg*nx][TAB] sweep table (rebuilt per species and stage)
    double* mom;         // [ns][11][nyg*nx] kept moments (+ max f as the 11th)
    double* gmom;        // [11][nx] moments of one edge row (ghost fill)
    double* bmark;       // [ns][2][11][g*nx] moments of the border rows at the marked time (section 4.1)
    double* bcur;        // [11][g*nx] the same rows now
    int bmark_valid;
    double* fields_stage;// [6][nyg*nx] device staging of E,B for vlasov_step_host
    int* errflag;        // device int: first asynchronous error
    int mom_valid;
    int fuse_xy;         // 1: use the fused spatial stage where it applies (vlasov_set_option)
    int fuse_mom;        // 1: VXV order: reduce the moments in the last vy+vz pass where that kernel can
    int64_t launches;
    int* h_err;          // pinned host mirror of errflag
    double* Jbuf;        // [3][nyg*nx] current density of vlasov_cycle
    double* Bavg;        // [3][nyg*nx] B at the E time level of vlasov_cycle
    // optional per-kernel timing (vlasov_timing_*): event pairs around every launch
    int timing;
    int ghost_tag;       // 1 while the launches being issued belong to the ghost fill / ghost rows (timing kinds)
    int nrec;
    static constexpr int MAX_REC = 8192;
    cudaEvent_t* ev0;    // [MAX_REC]
    cudaEvent_t* ev1;
    int* rec_kind;
};

namespace vl {

enum Kind { K_SWEEP_X = 0, K_SWEEP_Y, K_TABLE, K_VSWEEP_X, K_VSWEEP_YZ, K_MOMENTS, K_GHOST_TABLE, K_CURRENT,
            K_MAXWELL, K_SWEEP_XY, K_SWEEP_YX, K_GHOST_VSWEEP_X, K_GHOST_VSWEEP_YZ, K_GHOST_MOMENTS, K_GHOST_SWEEP_X,
            K_SWEEP_Z, K_COUNT };
static_assert((int)K_COUNT == (int)VLASOV_KIND_COUNT, "kinds of vlasov.h");

// Counts a launch and, when timing is on, brackets it with an event pair on the context's stream.
struct Launch {
    vlasov_ctx* c; int slot;
    Launch(vlasov_ctx* ctx, int kind) : c(ctx), slot(-1) {
        c->launches++;
        if (c->ghost_tag) {      // work that only exists because a side is FLUID gets its own kind
            if (kind == K_VSWEEP_X) kind = K_GHOST_VSWEEP_X;
            else if (kind == K_VSWEEP_YZ) kind = K_GHOST_VSWEEP_YZ;
            else if (kind == K_MOMENTS) kind = K_GHOST_MOMENTS;
            else if (kind == K_SWEEP_X) kind = K_GHOST_SWEEP_X;
        }
        if (c->timing && c->nrec < vlasov_ctx::MAX_REC) {
            slot = c->nrec++;
            c->rec_kind[slot] = kind;
            cudaEventRecord(c->ev0[slot], c->stream);
        }
    }
    ~Launch() { if (slot >= 0) cudaEventRecord(c->ev1[slot], c->stream); }
};

#define VL_CUDA_OK(call) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) return VLASOV_ECUDA; } while (0)

// ---- launchers (each returns VLASOV_OK / VLASOV_ECUDA and bumps ctx->launches) -----------------
// spatial half sweeps, out of place src -> dst (a1, a2, a7, a8 of DESIGN.md)
int launch_sweep_x(vlasov_ctx* c, const Species& s, const double* src, double* dst, double dts);
int launch_sweep_y(vlasov_ctx* c, const Species& s, const double* src, double* dst, double dts);
int launch_sweep_z(vlasov_ctx* c, const Species& s, const double* src, double* dst, double dts);   // 3D3V, periodic
// x sweep of rows [row0, row0+nrows) only (ghost rows beside a fused stage)
int launch_sweep_x_rows(vlasov_ctx* c, const Species& s, const double* src, double* dst, double dts, int row0, int nrows);
// fused spatial stage (sweep_space_fused.cu): x then y (xfirst) or y then x, interior rows, src -> dst
bool fused_xy_applicable(const vlasov_ctx* c, const Species& s, double dts);
int launch_sweep_xy(vlasov_ctx* c, const Species& s, const double* src, double* dst, double dts, int xfirst);
// Lorentz table (a3) and velocity sweeps (a4-a6), in place on f, rows [row0, row0+nrows)
int launch_lorentz_table(vlasov_ctx* c, const Species& s, const double* E, const double* B, double dt);
// ghost: the launch is a ghost fill (tiles read the edge cell T[16] and are scaled by T[15])
// mom_out: if not null, [11][nrows*nx] moments of the swept rows MAY be reduced in the same pass (*mom_done tells).
// src: if not null, the vx sweep reads src and writes f (out of place; vy and vz then run in place on f).
int launch_vsweeps(vlasov_ctx* c, const Species& s, double* f, int row0, int nrows, bool ghost = false,
                   double* mom_out = nullptr, bool* mom_done = nullptr, const double* src = nullptr);
// moments (a9): out[11][nyg*nx] (10 moments + max f) of rows [row0,row0+nrows) of f
int launch_moments(vlasov_ctx* c, const Species& s, const double* f, double* out, int row0, int nrows);
int species_max_f(vlasov_ctx* c, const Species& s, double* result);      // max f over all cells (synchronises)
// ghost fill (a0) of one side
int launch_ghost_fill(vlasov_ctx* c, const Species& s, double* f, int side);
int launch_lerp(vlasov_ctx* c, const double* a, const double* b, double theta, double* out, long n);
int launch_gather_rows(vlasov_ctx* c, const double* src, long src_stride, long off, double* dst, long n, int nk);
int launch_current(vlasov_ctx* c, double* J);
int launch_maxwell(vlasov_ctx* c, double dt, int nsub, double* E, double* B, const double* J, double* Bavg);

// ---- device helpers shared by all sweep kernels ------------------------------------------------
// Limited slopes of cell j, eqs. (43), (44) PAPER.md:273-276 with R6, written division-free:
//   eps+ (f_{j+1}-f_j) = clamp(d+, -max(0,Bv), max(0,A)),  eps- (f_j-f_{j-1}) = clamp(d-, -max(0,A), max(0,Bv)),
//   A = 2 f_j, Bv = 2 (f_inf - f_j).  Algebraically identical to the quotient form.
__device__ __forceinline__ void limited_slopes(double fm, double f0, double fp, double finf, int limiter,
                                               double& sp, double& sm) {
    double dp = fp - f0, dm = f0 - fm;
    if (limiter) {
        double A = f0 + f0;
        double Bv = 2.0 * (finf - f0);
        double hiA = fmax(A, 0.0), hiB = fmax(Bv, 0.0);
        sp = fmin(fmax(dp, -hiB), hiA);
        sm = fmin(fmax(dm, -hiA), hiB);
    } else {
        sp = dp; sm = dm;
    }
}

// Partial flux of the foot cell: b * [ f_j + (1-b)(2-b)/6 * eps+ d+ + (1-b)(1+b)/6 * eps- d- ],
// eq. (46) PAPER.md:288 (b = alpha in [0,1]); eq. (47) is the same expression on the mirrored line.
__device__ __forceinline__ double partial_flux(double fm, double f0, double fp, double b, double finf, int limiter) {
    double sp, sm;
    limited_slopes(fm, f0, fp, finf, limiter, sp, sm);
    double omb = 1.0 - b;
    double t = omb * (1.0 / 6.0);
    double c1 = t * (2.0 - b);
    double c2 = t * (1.0 + b);
    return b * (f0 + c1 * sp + c2 * sm);
}

// ---- shared memory by 32-bit address (keeps the window base out of the inner loops) ----------------
__device__ __forceinline__ double lds(unsigned a) {
    double v;
    asm volatile("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(a));
    return v;
}
__device__ __forceinline__ void sts(unsigned a, double v) { asm volatile("st.shared.f64 [%0], %1;" ::"r"(a), "d"(v)); }
__device__ __forceinline__ void cp_async8(unsigned dst, const double* src) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(dst), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }
__device__ __forceinline__ unsigned smem_addr(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }

// max(x, 0) on the bit pattern (no NaN fix-up code): x if its sign bit is clear, else +0.
__device__ __forceinline__ double relu_bits(double x) {
    const int h = __double2hiint(x);
    const int m = ~(h >> 31);
    return __hiloint2double(h & m, __double2loint(x) & m);
}

// Limited slopes eps+ d+, eps- d- of eqs. (43), (44) (R6) in the division-free clamp form
//     eps+ d+ = clamp(d+, -max(0,Bv), max(0,A)),  eps- d- = clamp(d-, -max(0,A), max(0,Bv)),  A = 2 f0, Bv = 2 (f_inf - f0)
// written in sign/magnitude: |eps d| = min(|d|, bound picked by the sign of d).  fp64 issue slots are the
// scarce resource on this path, so the test "does any lane of the warp
// need limiting at all" is done on the HIGH WORDS of the doubles in the integer pipe: for non-negative
// doubles the IEEE order is the integer order, so
//     hi(|d|) < min(hi(2 f0), hi(2 (f_inf - f0)))   ==>   |d| < min(2 f0, 2 (f_inf - f0))   ==>   eps = 1.
// The test is conservative (ties and negative bounds fall through to the exact clamps); hi(2 x) is
// hi(x) + 2^20 (exponent + 1; the denormal corner only ever errs by < 1e-307).
// FULL: the caller guarantees that all 32 lanes of the warp make this call (saves the active-mask bookkeeping).
template <int LIM, int FULL = 0>
__device__ __forceinline__ void slopes_fast(double fm, double f0, double fp, double finf, double& sp, double& sm) {
    const double dp = fp - f0, dm = f0 - fm;
    sp = dp; sm = dm;
    if (LIM) {
        const double g = finf - f0;
        const int hf = __double2hiint(f0) + 0x00100000, hg = __double2hiint(g) + 0x00100000;
        const int hp = __double2hiint(dp) & 0x7fffffff, hm = __double2hiint(dm) & 0x7fffffff;
        const int hmax = max(hp, hm);
        const unsigned mask = FULL ? 0xffffffffu : __activemask();
        if (__any_sync(mask, hmax >= min(hf, hg))) {
            const double hiA = relu_bits(f0 + f0);
            if (!__any_sync(mask, hmax >= hg)) {
                // only the positivity bound 2 f0 can bind (the tails of a distribution, far below f_inf):
                // eps+ d+ = min(d+, hiA), eps- d- = max(d-, -hiA)
                const double nA = -hiA;
                sp = dp < hiA ? dp : hiA;
                sm = dm > nA ? dm : nA;
            } else {
                const double hiB = relu_bits(g + g);
                const bool pneg = __double2hiint(dp) < 0, mneg = __double2hiint(dm) < 0;
                const double bp = pneg ? hiB : hiA;
                const double bm = mneg ? hiA : hiB;
                const double ap = __hiloint2double(hp, __double2loint(dp));      // |d+|
                const double am = __hiloint2double(hm, __double2loint(dm));      // |d-|
                const double mp = ap < bp ? ap : bp;
                const double mm = am < bm ? am : bm;
                sp = __hiloint2double(__double2hiint(mp) | (__double2hiint(dp) & 0x80000000), __double2loint(mp));
                sm = __hiloint2double(__double2hiint(mm) | (__double2hiint(dm) & 0x80000000), __double2loint(mm));
            }
        }
    }
}

// The exact clamps of slopes_fast (both bounds), applied in place to the raw differences sp = d+, sm = d- of a cell
// with value f0: |eps d| = min(|d|, bound picked by the sign of d), sign restored.
__device__ __forceinline__ void slopes_exact(double f0, double finf, double& sp, double& sm) {
    const double dp = sp, dm = sm, g = finf - f0;
    const double hiA = relu_bits(f0 + f0), hiB = relu_bits(g + g);
    const int hp = __double2hiint(dp) & 0x7fffffff, hm = __double2hiint(dm) & 0x7fffffff;
    const bool pneg = __double2hiint(dp) < 0, mneg = __double2hiint(dm) < 0;
    const double bp = pneg ? hiB : hiA;
    const double bm = mneg ? hiA : hiB;
    const double ap = __hiloint2double(hp, __double2loint(dp));      // |d+|
    const double am = __hiloint2double(hm, __double2loint(dm));      // |d-|
    const double mp = ap < bp ? ap : bp;
    const double mm = am < bm ? am : bm;
    sp = __hiloint2double(__double2hiint(mp) | (__double2hiint(dp) & 0x80000000), __double2loint(mp));
    sm = __hiloint2double(__double2hiint(mm) | (__double2hiint(dm) & 0x80000000), __double2loint(mm));
}

// n = floor(s) for s >= 0 up to the exact-integer case, where n = s - 1, b = 1 is returned instead:
// the flux is identical there (R8).  Magic-number rounding, no conversion-pipe instruction.
__device__ __forceinline__ void split_shift(double s, int& n, double& b) {
    const double M = 6755399441055744.0;   // 1.5 * 2^52
    double r = (s - 0.5) + M;
    n = __double2loint(r);
    b = s - (r - M);
}

}  // namespace vl
