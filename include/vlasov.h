/* vlasov.h -- C ABI of the B200-native Vlasov full-step hot path of arXiv 1406.5445
 * (Rieke, Trost, Grauer, "Coupled Vlasov and two-fluid codes on GPUs").
 *
 * Citations are PAPER.md:<line> plus the section / equation they fall in.  Readings R1..R21 of the
 * garbled or silent passages are listed in DESIGN.md.
 *
 * Conventions (all entry points):
 *   - every pointer named *_dev is DEVICE memory owned by the caller (a torch allocation), fp64,
 *     128-byte aligned; pointers without the suffix are HOST memory read during the call only;
 *   - the library keeps the device pointers handed to vlasov_init (no copies): they must outlive
 *     the context;
 *   - all work is enqueued on cfg.stream (a cudaStream_t) and returns asynchronously;
 *   - every call returns an int: 0 = ok, negative = error; nothing throws, nothing prints;
 *   - data-dependent failures (VLASOV_ESHIFT, VLASOV_EDOMAIN) are recorded in a device flag and
 *     surfaced by vlasov_check, which synchronises the stream;
 *   - there is no CPU fallback: without a CUDA device vlasov_init returns VLASOV_ECUDA.
 *
 * Data layout:
 *   f_s      [ny_g][nx][nvx][nvy][nvz]   cell averages (R1), velocity fastest, ny_g = ny + 2 nghost_y
 *   E, B, J  [3][ny_g][nx]
 *   moments  [10][ny_g][nx] = M0, M1x, M1y, M1z, M2xx, M2yy, M2zz, M2xy, M2xz, M2yz
 *   3D3V (cfg.nz > 1): f_s [nz][ny][nx][nvx][nvy][nvz], E, B, J [3][nz][ny][nx], moments [10][nz][ny][nx]; the step
 *   is x/2 y/2 z/2 - vx vy vz - z/2 y/2 x/2 (XVX) or v/2 - x y z - v/2 (VXV); fields on the 3D Yee grid (R24)
 *   fluid5   [5][nghost_y][nx] = n, ux, uy, uz, p; ghost layer index counted OUTWARD from the edge
 */
#ifndef VLASOV_B200_H
#define VLASOV_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct vlasov_ctx vlasov_ctx; /* opaque */

enum {
    VLASOV_OK = 0,
    VLASOV_EINVAL = -1,  /* bad argument (null pointer, non-positive size, unknown enum) */
    VLASOV_EALIGN = -2,  /* a device pointer is not 128-byte aligned */
    VLASOV_ESHIFT = -3,  /* a y-shift reaches beyond the ghost rows of a FLUID side (R9) */
    VLASOV_EDOMAIN = -4, /* Boris denominator <= 0 (R13), or n<=0 / T<=0 / p<=0 in the ghost fill */
    VLASOV_ECUDA = -5,   /* a CUDA runtime call failed (or no device) */
    VLASOV_ETOOBIG = -6  /* vlasov_fluid_step_static: the block needs more than VLASOV_FLUID_STATIC_SCRATCH_BYTES */
};

/* y-side kinds; x is always periodic (R16, R19). */
enum { VLASOV_BC_PERIODIC = 0, VLASOV_BC_REFLECT = 1, VLASOV_BC_FLUID = 2 };

/* Strang order: eq. (22) PAPER.md:154 (default) or the order of the coupled cycle, PAPER.md:420 (R2). */
enum { VLASOV_ORDER_XVX = 0, VLASOV_ORDER_VXV = 1 };

/* Stage mask of vlasov_step.  XVX: X1 = x/2 then y/2, V = vx,vy,vz, X2 = y/2 then x/2 (R3).
 * VXV: X1 = first velocity half, V = full spatial step (x then y), X2 = second velocity half. */
enum {
    VLASOV_STAGE_X1 = 1,
    VLASOV_STAGE_V = 2,
    VLASOV_STAGE_X2 = 4,
    VLASOV_STAGE_GHOST = 8,    /* ghost fill of FLUID sides, section 4.2 */
    VLASOV_STAGE_MOMENTS = 16, /* moments of the final f, kept for vlasov_moments / vlasov_current */
    VLASOV_STAGE_ALL = 31
};

typedef struct {
    double q, m;       /* charge and mass, eq. (1) */
    int32_t nv[3];     /* velocity cells per direction (any; an even nv[2] takes the 16-byte paths) */
    double vmin[3];    /* lower faces of the velocity box; centres vmin + (k+1/2) dv */
    double vmax[3];    /* upper faces */
    double f_inf;      /* f_infinity of eqs. (43),(44) PAPER.md:273-276 (R6): a per-species upper bound of f, > 0;
                          <= 0: vlasov_init takes max f of the species' f_dev as it stands (one pass, synchronises) */
} vlasov_species;

typedef struct {
    int32_t nx, ny;       /* interior spatial cells */
    int32_t nghost_y;     /* ghost rows per y side (R16); 0 unless a side is FLUID */
    int32_t nspecies;
    double lx, ly;        /* extent of the interior block: dx = lx/nx, dy = ly/ny */
    int32_t bc_y_lo, bc_y_hi;
    int32_t order;        /* VLASOV_ORDER_* */
    int32_t limiter;      /* 1 = eqs. (43),(44); 0 = eps == 1 (unlimited third order) */
    int32_t fields_yee;   /* 0: E,B,J cell-centred; 1: Yee positions of R17 / R24 */
    int32_t nz;           /* 3D3V (NEXT-4): cells along z, periodic; 0 or 1 = the 2D3V path.  nz > 1 needs
                             nghost_y == 0 (no FLUID sides) and lz > 0; every array gains a slowest index iz */
    double c, mu0;        /* Maxwell constants, eqs. (9),(10) PAPER.md:68-71 */
    double lz;            /* extent along z: dz = lz/nz (ignored for nz <= 1) */
    void* stream;         /* cudaStream_t; NULL = legacy default stream */
} vlasov_config;

/* Bytes of device scratch vlasov_init needs: one ping-pong copy of the largest species' f, the
 * per-spatial-cell sweep tables and the kept moments.  Returns 0 on invalid arguments. */
size_t vlasov_scratch_bytes(const vlasov_config* cfg, const vlasov_species* sp /*[nspecies]*/);

/* Create a context.  f_dev[s] points at species s' phase-space array (layout above).
 * A REFLECT side needs a vy grid that is symmetric about 0 (vmin[1] == -vmax[1], R19): the wall image is built by
 * mirroring the i_vy index.
 * Errors: EINVAL (also: asymmetric vy grid with a REFLECT side), EALIGN, ECUDA.  *out is NULL on error. */
int vlasov_init(const vlasov_config* cfg, const vlasov_species* sp /*[nspecies]*/,
                double* const* f_dev /*[nspecies], host array of device pointers*/,
                void* scratch_dev, size_t scratch_bytes, vlasov_ctx** out);

/* Kind of one y side of one species and, for FLUID, the 5-moment fluid state of its ghost cells
 * (section 4.2, summary PAPER.md:399-402; eq. (8) PAPER.md:61 turns p into the target temperature).
 * The pointer is kept and read at the next vlasov_step with STAGE_GHOST.  side: 0 = y_lo, 1 = y_hi.
 * kind must equal cfg.bc_y_lo / bc_y_hi of that side.  Errors: EINVAL. */
int vlasov_set_boundary(vlasov_ctx* ctx, int species, int side, int kind, const double* fluid5_dev);

/* One full step of eq. (1) for every species: Strang splitting eq. (22), 1D PFC
 * remaps eqs. (38), (43)-(47) PAPER.md:247-295, velocity sweeps by backsubstitution eqs. (33)-(35)
 * PAPER.md:212-227 in the order vx, vy, vz.  E_dev, B_dev are the time-centred
 * fields, held fixed over the step (R11).  f is updated in the caller's buffers.
 * Errors: EINVAL (also: STAGE_GHOST with a FLUID side whose fluid state was never given to vlasov_set_boundary);
 * ESHIFT / EDOMAIN asynchronously (vlasov_check). */
int vlasov_step(vlasov_ctx* ctx, double dt, const double* E_dev, const double* B_dev, uint32_t stages);

/* The same step driven from HOST buffers, the way the paper's cycle crosses the CPU/GPU border
 * (Maxwell and fluid solvers on the CPUs, Vlasov on the GPUs): E_host, B_host
 * ([3][ny_g][nx], pinned or pageable) are copied to the device, the step runs, and if mom_host is not
 * NULL the moments of all species ([nspecies][10][ny_g][nx]) are copied back.  Synchronises the
 * stream; returns like vlasov_check.  f stays resident on the device. */
int vlasov_step_host(vlasov_ctx* ctx, double dt, const double* E_host, const double* B_host, uint32_t stages,
                     double* mom_host);

/* Raw velocity moments of species s, eqs. (2)-(4) PAPER.md:39-46 as midpoint sums times dv^3 (R14).
 * If the last vlasov_step on this context ran STAGE_MOMENTS and f has not been touched since
 * (vlasov_touch), the kept result is copied; otherwise f is reduced again. */
int vlasov_moments(vlasov_ctx* ctx, int species, double* mom_dev /*[10][ny_g][nx]*/);

/* Boundary data for the two-fluid code, section 4.1: "the boundary data needed by the two-fluid code
 * can be calculated by means of the moment equations (2)-(4) ... needs boundary conditions at times t, t + dt/2 and
 * t + dt.  Thus the Vlasov data has to be advanced before the fluid data.  Then, by linear interpolation in time, the
 * intermediate boundary conditions can be calculated".
 * vlasov_fluid_boundary_mark: call at time t, before the step: keeps the raw moments (layout and order of
 *   vlasov_moments) of the nghost_y interior rows next to both y borders, for every species (reading R22: the fluid
 *   block's ghost cells are as deep as the kinetic block's).
 * vlasov_fluid_boundary: call after the step: reduces the same rows of the current f and writes
 *   (1 - theta) * marked + theta * current to out_dev [10][nghost_y][nx] (row l = l-th of those rows in ascending y;
 *   side 0 = y_lo: interior rows 0..g-1, side 1 = y_hi: interior rows ny-g..ny-1).  theta in [0,1] is not enforced
 *   (extrapolation is the caller's business).
 * Errors: EINVAL (nghost_y == 0, ny < nghost_y, bad species/side, no mark yet, NULL), EALIGN. */
int vlasov_fluid_boundary_mark(vlasov_ctx* ctx);
int vlasov_fluid_boundary(vlasov_ctx* ctx, int species, int side, double theta, double* out_dev /*[10][g][nx]*/);

/* Current density j = sum_s q_s M1^(s), eq. (11), at cell centres or (fields_yee)
 * linearly interpolated to the E positions of R17. */
int vlasov_current(vlasov_ctx* ctx, double* J_dev /*[3][ny_g][nx]*/);

/* nsub FDTD leapfrog sub-steps of dt/nsub on the 2D Yee grid (section 3.3, eqs. (9),
 * (10); cycle PAPER.md:419,423): E += ddt c^2 (curl B - mu0 J), then B -= ddt curl E; J held fixed.
 * On entry B is half a sub-step ahead of E.  Bavg_dev (may be NULL) receives B linearly interpolated
 * to the final time of E.  y walls are PEC unless bc_y_lo is PERIODIC. */
int vlasov_maxwell(vlasov_ctx* ctx, double dt, int nsub, double* E_dev, double* B_dev,
                   const double* J_dev, double* Bavg_dev);

/* One cycle of section 4.3 (Fig. 2) without the fluid step (item 4, out
 * of scope): currents (eq. 11) -> fields half a step (nsub sub-steps of dt/(2 nsub)) -> one complete
 * Vlasov step with the new E and with B interpolated to the E time level -> currents ->
 * fields another half step.  E_dev, B_dev ([3][ny_g][nx]) are advanced in place; stages = ALL. */
int vlasov_cycle(vlasov_ctx* ctx, double dt, int nsub, double* E_dev, double* B_dev);

/* vlasov_cycle from HOST buffers (the paper's CPU-side Maxwell/fluid data): E_host,
 * B_host are copied in, advanced, and copied back; mom_host (may be NULL) receives the moments of all
 * species [nspecies][10][ny_g][nx].  Synchronises; returns like vlasov_check. */
int vlasov_cycle_host(vlasov_ctx* ctx, double dt, int nsub, double* E_host, double* B_host, double* mom_host);

/* Per-kernel device timing for the roofline report: while enabled every launch is bracketed by a
 * CUDA event pair on the stream.  vlasov_timing_read synchronises, sums milliseconds and launch
 * counts per kernel kind (VLASOV_KIND_*) into host arrays of length >= VLASOV_KIND_COUNT, and
 * clears the record. */
enum {
    VLASOV_KIND_SWEEP_X = 0, VLASOV_KIND_SWEEP_Y, VLASOV_KIND_TABLE, VLASOV_KIND_VSWEEP_X, VLASOV_KIND_VSWEEP_YZ,
    VLASOV_KIND_MOMENTS, VLASOV_KIND_GHOST_TABLE, VLASOV_KIND_CURRENT, VLASOV_KIND_MAXWELL, VLASOV_KIND_SWEEP_XY /* fused x/2 y/2 */,
    VLASOV_KIND_SWEEP_YX /* fused y/2 x/2 */,
    /* launches that only exist because a side is FLUID (config 4's "ghost-fill share of step time"): the ghost fill's
     * velocity remaps and edge-row moments (section 4.2), and the x sweeps of the ghost rows beside a fused stage */
    VLASOV_KIND_GHOST_VSWEEP_X, VLASOV_KIND_GHOST_VSWEEP_YZ, VLASOV_KIND_GHOST_MOMENTS, VLASOV_KIND_GHOST_SWEEP_X,
    VLASOV_KIND_SWEEP_Z /* 3D3V: the third spatial sweep */,
    VLASOV_KIND_COUNT
};
int vlasov_timing_enable(vlasov_ctx* ctx, int on);
int vlasov_timing_read(vlasov_ctx* ctx, double* ms_by_kind, int64_t* count_by_kind, int nkinds);

/* Execution options (results stay within the parity tolerance either way).
 * VLASOV_OPT_FUSE_XY (default 1): run each spatial stage (x/2 y/2, y/2 x/2) as ONE fused pass over f when every
 * shift of the stage is below one cell; 0 = always the general one-direction kernels.  Errors: EINVAL.
 * VLASOV_OPT_FUSE_MOMENTS (default 1): ORDER_VXV only: reduce the moments of the final f inside the last
 * velocity pass (vy+vz kernel, 16^3 / 32^3 velocity blocks) instead of a separate pass over f; 0 = always the separate
 * moments kernel. */
enum { VLASOV_OPT_FUSE_XY = 1, VLASOV_OPT_FUSE_MOMENTS = 2 };
int vlasov_set_option(vlasov_ctx* ctx, int option, int value);

/* Tell the library the caller wrote into an f buffer itself (drops the kept moments). */
int vlasov_touch(vlasov_ctx* ctx);

/* Synchronise the stream; return the first asynchronously recorded error (and clear it). */
int vlasov_check(vlasov_ctx* ctx);

/* Number of kernels this context has launched since vlasov_init (bench.py's gpu_launches). */
int64_t vlasov_launch_count(const vlasov_ctx* ctx);

void vlasov_free(vlasov_ctx* ctx);
const char* vlasov_strerror(int err);

/* ---- the fluid side of the coupling (section 3.2; cycle item 4 PAPER.md:421) ----------
 * Five-moment fluid step per species: the moment equations (5)-(7) PAPER.md:50-54 with the adiabatic closure (8)
 * PAPER.md:61 and the Lorentz source, "CWENO scheme [18] ... third order strong-stability-preserving Runge-Kutta scheme
 * by Shu and Osher [19]" (details: reading R23 of DESIGN.md).  Stateless: no context, every array is the caller's.
 *   U_dev      [nspecies][5][ny + 4][nx]  cell averages of rho, u_x, u_y, u_z (MOMENTUM density, eq. 3), energy density;
 *              two ghost rows per y side (scratch unless the side is COUPLED ... and then they are overwritten too)
 *   E_dev, B_dev  [3][ny + 4][nx]  fields at the cell centres, held fixed over the step
 *   ghost_lo_dev, ghost_hi_dev  [3][nspecies][5][2][nx]  ghost rows (ascending y) of a COUPLED side at the three
 *              Runge-Kutta stage times t, t + dt, t + dt/2 -- in this order (section 4.1: "needs boundary
 *              conditions at times t, t + dt/2 and t + dt ... by linear interpolation in time"); NULL for other kinds
 * x is periodic.  Errors: EINVAL, EALIGN, ECUDA. */
enum { VLASOV_FLUID_BC_PERIODIC = 0, VLASOV_FLUID_BC_WALL = 1 /* mirror image, u_y odd */, VLASOV_FLUID_BC_COUPLED = 2 };
enum { VLASOV_FLUID_MAX_SPECIES = 8 };
typedef struct {
    int32_t nx, ny;          /* interior cells of the fluid block */
    int32_t nspecies;
    int32_t bc_y_lo, bc_y_hi;
    int32_t reserved;
    double dx, dy;
    double q[VLASOV_FLUID_MAX_SPECIES], m[VLASOV_FLUID_MAX_SPECIES];
    void* stream;            /* cudaStream_t */
} vlasov_fluid_config;
size_t vlasov_fluid_scratch_bytes(const vlasov_fluid_config* cfg);
int vlasov_fluid_step(const vlasov_fluid_config* cfg, double dt, double* U_dev, const double* E_dev, const double* B_dev,
                      const double* ghost_lo_dev, const double* ghost_hi_dev, void* scratch_dev, size_t scratch_bytes);
/* vlasov_fluid_step for callers that cannot allocate device memory (code under CUDA graph capture, serving loops,
 * harnesses that forbid cudaMalloc): the same step, same arguments and results bit for bit, with the two Runge-Kutta
 * stage buffers in a file-scope `static __device__` array of the library instead of the caller's scratch_dev.  Calls no
 * cudaMalloc, cudaFree or allocating library routine; the array (VLASOV_FLUID_STATIC_SCRATCH_BYTES = 4 MiB, aligned to
 * 256 bytes) is part of the library image, so every GPU that loads the library holds it until the process exits.  Its
 * device address is looked up once per device (cudaGetSymbolAddress with that device current) on the first call there:
 * make one call per device outside any capture, with the device current that owns U_dev.
 *   Limit: vlasov_fluid_scratch_bytes(cfg) <= VLASOV_FLUID_STATIC_SCRATCH_BYTES, i.e. nspecies * (ny + 4) * nx <= 52428
 *   cells (e.g. 2 species on 256 x 98; the 256 x 48 blocks beside config 4's band need 2.1 MB); beyond it the call
 *   returns VLASOV_ETOOBIG and launches nothing.
 *   Sharing: every call on a device uses the same array, which keeps the last call's contents.  Nothing in it has to
 *   start at zero (each stage buffer is written in full, ghost rows included, before it is read), so nothing is cleared.
 *   Calls that overlap on the GPU (two streams, two host threads, this entry point inside two graphs that run
 *   concurrently) RACE on the array: serialise them, or use vlasov_fluid_step with scratch of your own.
 * Errors: those of vlasov_fluid_step, and ETOOBIG. */
#define VLASOV_FLUID_STATIC_SCRATCH_BYTES (4u << 20)
int vlasov_fluid_step_static(const vlasov_fluid_config* cfg, double dt, double* U_dev, const double* E_dev,
                             const double* B_dev, const double* ghost_lo_dev, const double* ghost_hi_dev);
/* eqs. (2)-(4) PAPER.md:39-46: rho = m M0, u = m M1, energy = (m/2)(M2xx + M2yy + M2zz) from raw moments [10][n] (the
 * layout of vlasov_moments / vlasov_fluid_boundary) to fluid variables [5][n]. */
int vlasov_fluid_from_moments(const double* mom10_dev, double m, double* U5_dev, long n, void* stream);
/* eq. (8): fluid variables [5][n] to what vlasov_set_boundary takes, [5][n] = n, bulk velocity, pressure. */
int vlasov_fluid_to_boundary(const double* U5_dev, double m, double* fluid5_dev, long n, void* stream);

#ifdef __cplusplus
}
#endif
#endif /* VLASOV_B200_H */
