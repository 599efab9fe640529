// C ABI of libvlasov_b200 (include/vlasov.h): argument checks, scratch carve-up, and the host-side
// sequencing of one Vlasov step (Strang splitting eq. (22); cycle of section 4.3
// PAPER.md:418-423).  Every arithmetic step of the path runs in the kernels of this directory.
#include <new>
#include "vlasov_internal.cuh"

using namespace vl;

namespace {

inline size_t align_up(size_t x) { return (x + 127) & ~(size_t)127; }

struct Carve {
    size_t pong, table, mom, gmom, bmark, bcur, fields, jbuf, bavg, err, total;
};

bool carve(const vlasov_config* cfg, const vlasov_species* sp, Carve& C) {
    if (!cfg || !sp) return false;
    if (cfg->nx <= 0 || cfg->ny <= 0 || cfg->nghost_y < 0 || cfg->nspecies <= 0 || cfg->nspecies > MAX_SPECIES) return false;
    const size_t nyg = (size_t)cfg->ny + 2 * (size_t)cfg->nghost_y;
    const size_t ncell = nyg * cfg->nx * (size_t)(cfg->nz > 1 ? cfg->nz : 1);
    size_t maxS = 0;
    for (int s = 0; s < cfg->nspecies; ++s) {
        if (sp[s].nv[0] <= 0 || sp[s].nv[1] <= 0 || sp[s].nv[2] <= 0) return false;
        size_t S = (size_t)sp[s].nv[0] * sp[s].nv[1] * sp[s].nv[2];
        if (S > maxS) maxS = S;
    }
    size_t off = 0;
    C.pong = off;   off += align_up(maxS * ncell * 8);
    C.table = off;  off += align_up(ncell * TAB * 8);
    C.mom = off;    off += align_up((size_t)cfg->nspecies * 11 * ncell * 8);
    C.gmom = off;   off += align_up((size_t)11 * cfg->nx * 8);
    C.bmark = off;  off += align_up((size_t)cfg->nspecies * 2 * 11 * cfg->nghost_y * cfg->nx * 8);
    C.bcur = off;   off += align_up((size_t)11 * cfg->nghost_y * cfg->nx * 8);
    C.fields = off; off += align_up(6 * ncell * 8);
    C.jbuf = off;   off += align_up(3 * ncell * 8);
    C.bavg = off;   off += align_up(3 * ncell * 8);
    C.err = off;    off += 128;
    C.total = off;
    return true;
}

int species_step(vlasov_ctx* c, int si, double dt, const double* E, const double* B, uint32_t stages) {
    Species& s = c->sp[si];
    const Geom& G = c->G;
    int e;
    if (stages & VLASOV_STAGE_GHOST) {
        c->ghost_tag = 1;
        e = VLASOV_OK;
        if (G.bc_lo == VLASOV_BC_FLUID) e = launch_ghost_fill(c, s, s.f, 0);
        if (!e && G.bc_hi == VLASOV_BC_FLUID) e = launch_ghost_fill(c, s, s.f, 1);
        c->ghost_tag = 0;
        if (e) return e;
    }
    // cur: where this species' f lives right now.  The general spatial stage is f -> pong -> f; the fused
    // stage is ONE pass cur -> other, so the buffers swap roles; an odd number of fused stages in one call
    // is settled by a copy back into the caller's buffer at the end.
    double* cur = s.f;
    auto other_of = [&](double* p) { return p == s.f ? c->pong : s.f; };
    // x and y half sweeps of one spatial stage (every z slab), src = cur; leaves the result in cur
    auto space_xy = [&](double dts, bool x_first) -> int {
        int r;
        double* other = other_of(cur);
        if (c->fuse_xy && fused_xy_applicable(c, s, dts)) {
            r = launch_sweep_xy(c, s, cur, other, dts, x_first ? 1 : 0); if (r) return r;
            if (G.g > 0) {      // x sweeps update ghost rows too, y sweeps never do (R16)
                c->ghost_tag = 1;
                r = launch_sweep_x_rows(c, s, cur, other, dts, 0, G.g);
                if (!r) r = launch_sweep_x_rows(c, s, cur, other, dts, G.g + G.ny, G.g);
                c->ghost_tag = 0;
                if (r) return r;
            }
            cur = other;
            return VLASOV_OK;
        }
        if (x_first) {
            r = launch_sweep_x(c, s, cur, other, dts); if (r) return r;
            return launch_sweep_y(c, s, other, cur, dts);
        }
        r = launch_sweep_y(c, s, cur, other, dts); if (r) return r;
        return launch_sweep_x(c, s, other, cur, dts);
    };
    auto space_z = [&](double dts) -> int {          // 3D3V: the third spatial sweep, out of place
        if (G.nz <= 1) return VLASOV_OK;
        double* other = other_of(cur);
        int r = launch_sweep_z(c, s, cur, other, dts); if (r) return r;
        cur = other;
        return VLASOV_OK;
    };
    // forward: x y z (before the velocity step); backward: z y x (palindrome, R3)
    auto space = [&](double dts, bool forward) -> int {
        int r;
        if (forward) { r = space_xy(dts, true); if (r) return r; return space_z(dts); }
        r = space_z(dts); if (r) return r;
        return space_xy(dts, false);
    };
    bool mom_done = false;
    // flips_after: how many fused (one pass, buffer-swapping) spatial stages still follow in this call.  The vx sweep
    // can read one buffer and write the other, so the velocity step is where f changes sides for free: it leaves f
    // where the remaining stages bring it home to the caller's buffer without a copy.
    auto velocity = [&](double dtv, int flips_after, bool with_moments = false) -> int {
        int r = launch_lorentz_table(c, s, E, B, dtv); if (r) return r;
        double* target = (flips_after & 1) ? c->pong : s.f;
        // with_moments (the last pass of a VXV step): the moments of the final f may be reduced by the vy+vz kernel
        // itself.  All rows, ghost rows too (R16).
        double* mo = with_moments && c->fuse_mom && target == s.f ? c->mom + (long)si * 11 * ((long)G.nrows * G.nx) : nullptr;
        r = launch_vsweeps(c, s, target, 0, G.nrows, false, mo, &mom_done, cur);
        cur = target;
        return r;
    };
    // buffer changes of one spatial stage: the fused x,y pass (one) and the z sweep (one)
    auto flips = [&](bool requested, double dts) {
        return !requested ? 0 : (c->fuse_xy && fused_xy_applicable(c, s, dts) ? 1 : 0) + (G.nz > 1 ? 1 : 0);
    };
    if (c->order == VLASOV_ORDER_XVX) {
        if (stages & VLASOV_STAGE_X1) { e = space(dt / 2.0, true); if (e) return e; }
        if (stages & VLASOV_STAGE_V) { e = velocity(dt, flips((stages & VLASOV_STAGE_X2) != 0, dt / 2.0)); if (e) return e; }
        if (stages & VLASOV_STAGE_X2) { e = space(dt / 2.0, false); if (e) return e; }     // palindrome, R3
    } else {
        if (stages & VLASOV_STAGE_X1) { e = velocity(dt / 2.0, flips((stages & VLASOV_STAGE_V) != 0, dt)); if (e) return e; }
        if (stages & VLASOV_STAGE_V) { e = space(dt, true); if (e) return e; }
        if (stages & VLASOV_STAGE_X2) { e = velocity(dt / 2.0, 0, (stages & VLASOV_STAGE_MOMENTS) != 0); if (e) return e; }
    }
    if (cur != s.f) {
        VL_CUDA_OK(cudaMemcpyAsync(s.f, cur, (size_t)G.nrows * G.nx * s.nvtot * 8, cudaMemcpyDeviceToDevice, c->stream));
        c->launches++;
    }
    if ((stages & VLASOV_STAGE_MOMENTS) && !mom_done) {
        const long ncell = (long)G.nrows * G.nx;
        e = launch_moments(c, s, s.f, c->mom + (long)si * 11 * ncell, 0, G.nrows); if (e) return e;
    }
    return VLASOV_OK;
}

int ensure_moments(vlasov_ctx* c) {
    if (c->mom_valid) return VLASOV_OK;
    const long ncell = (long)c->G.nrows * c->G.nx;
    for (int s = 0; s < c->ns; ++s) {
        int e = launch_moments(c, c->sp[s], c->sp[s].f, c->mom + (long)s * 11 * ncell, 0, c->G.nrows);
        if (e) return e;
    }
    c->mom_valid = 1;
    return VLASOV_OK;
}

}  // namespace

extern "C" {

size_t vlasov_scratch_bytes(const vlasov_config* cfg, const vlasov_species* sp) {
    Carve C;
    return carve(cfg, sp, C) ? C.total : 0;
}

int vlasov_init(const vlasov_config* cfg, const vlasov_species* sp, double* const* f_dev, void* scratch_dev,
                size_t scratch_bytes, vlasov_ctx** out) {
    if (out) *out = nullptr;
    Carve C;
    if (!out || !f_dev || !scratch_dev || !carve(cfg, sp, C)) return VLASOV_EINVAL;
    if (scratch_bytes < C.total) return VLASOV_EINVAL;
    if (!(cfg->lx > 0.0) || !(cfg->ly > 0.0)) return VLASOV_EINVAL;
    if (cfg->bc_y_lo < 0 || cfg->bc_y_lo > 2 || cfg->bc_y_hi < 0 || cfg->bc_y_hi > 2) return VLASOV_EINVAL;
    if ((cfg->bc_y_lo == VLASOV_BC_PERIODIC) != (cfg->bc_y_hi == VLASOV_BC_PERIODIC)) return VLASOV_EINVAL;
    if ((cfg->bc_y_lo == VLASOV_BC_FLUID || cfg->bc_y_hi == VLASOV_BC_FLUID) && cfg->nghost_y < 1) return VLASOV_EINVAL;
    if (cfg->order != VLASOV_ORDER_XVX && cfg->order != VLASOV_ORDER_VXV) return VLASOV_EINVAL;
    if (cfg->nz < 0) return VLASOV_EINVAL;
    if (cfg->nz > 1 && (cfg->nghost_y != 0 || !(cfg->lz > 0.0))) return VLASOV_EINVAL;       // 3D3V: no ghost rows
    if (((uintptr_t)scratch_dev) & 127) return VLASOV_EALIGN;
    for (int s = 0; s < cfg->nspecies; ++s) {
        if (!f_dev[s]) return VLASOV_EINVAL;
        if (((uintptr_t)f_dev[s]) & 127) return VLASOV_EALIGN;
        if (!(sp[s].m > 0.0) || !(sp[s].f_inf == sp[s].f_inf)) return VLASOV_EINVAL;
        for (int d = 0; d < 3; ++d) if (!(sp[s].vmax[d] > sp[s].vmin[d])) return VLASOV_EINVAL;
        // a REFLECT wall builds its image by mirroring the i_vy index (R19): that is f(-vy) only on a symmetric vy grid
        if (cfg->bc_y_lo == VLASOV_BC_REFLECT || cfg->bc_y_hi == VLASOV_BC_REFLECT) {
            const double width = sp[s].vmax[1] - sp[s].vmin[1];
            const double skew = sp[s].vmin[1] + sp[s].vmax[1];
            if (!((skew < 0 ? -skew : skew) <= 1e-12 * width)) return VLASOV_EINVAL;
        }
    }
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev <= 0) return VLASOV_ECUDA;

    vlasov_ctx* c = new (std::nothrow) vlasov_ctx();
    if (!c) return VLASOV_ECUDA;
    c->G.nx = cfg->nx; c->G.ny = cfg->ny; c->G.g = cfg->nghost_y; c->G.nyg = cfg->ny + 2 * cfg->nghost_y;
    c->G.dx = cfg->lx / cfg->nx; c->G.dy = cfg->ly / cfg->ny;
    c->G.nz = cfg->nz > 1 ? cfg->nz : 1;
    c->G.nrows = c->G.nz * c->G.nyg;
    c->G.dz = c->G.nz > 1 ? cfg->lz / cfg->nz : 1.0;
    c->G.bc_lo = cfg->bc_y_lo; c->G.bc_hi = cfg->bc_y_hi;
    c->G.limiter = cfg->limiter ? 1 : 0; c->G.fields_yee = cfg->fields_yee ? 1 : 0;
    c->G.wall = cfg->bc_y_lo == VLASOV_BC_PERIODIC ? 0 : 1;
    c->order = cfg->order; c->c = cfg->c; c->mu0 = cfg->mu0;
    c->ns = cfg->nspecies;
    c->stream = (cudaStream_t)cfg->stream;
    for (int s = 0; s < c->ns; ++s) {
        Species& S = c->sp[s];
        S.q = sp[s].q; S.m = sp[s].m; S.f_inf = sp[s].f_inf;
        S.nvtot = 1;
        for (int d = 0; d < 3; ++d) {
            S.nv[d] = sp[s].nv[d]; S.vmin[d] = sp[s].vmin[d];
            S.dv[d] = (sp[s].vmax[d] - sp[s].vmin[d]) / sp[s].nv[d];
            S.nvtot *= sp[s].nv[d];
        }
        S.f = f_dev[s];
        S.fluid[0] = S.fluid[1] = nullptr;
    }
    char* base = (char*)scratch_dev;
    c->pong = (double*)(base + C.pong);
    c->table = (double*)(base + C.table);
    c->mom = (double*)(base + C.mom);
    c->gmom = (double*)(base + C.gmom);
    c->bmark = (double*)(base + C.bmark);
    c->bcur = (double*)(base + C.bcur);
    c->bmark_valid = 0;
    c->fields_stage = (double*)(base + C.fields);
    c->Jbuf = (double*)(base + C.jbuf);
    c->Bavg = (double*)(base + C.bavg);
    c->errflag = (int*)(base + C.err);
    c->timing = 0; c->ghost_tag = 0; c->nrec = 0; c->ev0 = c->ev1 = nullptr; c->rec_kind = nullptr;
    c->mom_valid = 0;
    c->fuse_xy = 1;
    c->fuse_mom = 1;
    c->launches = 0;
    c->h_err = nullptr;
    if (cudaMallocHost((void**)&c->h_err, sizeof(int)) != cudaSuccess) { delete c; return VLASOV_ECUDA; }
    if (cudaMemsetAsync(c->errflag, 0, 128, c->stream) != cudaSuccess) { cudaFreeHost(c->h_err); delete c; return VLASOV_ECUDA; }
    // f_inf <= 0: "take max f at init" (reading R6: f_infinity is an upper bound of f) -- one reduction
    // pass over the species' f as it stands now
    for (int s = 0; s < c->ns; ++s) {
        if (c->sp[s].f_inf > 0.0) continue;
        double mx = 0.0;
        const int e = species_max_f(c, c->sp[s], &mx);
        if (e || !(mx > 0.0)) { cudaFreeHost(c->h_err); delete c; return e ? e : VLASOV_EINVAL; }
        c->sp[s].f_inf = mx;
    }
    c->launches = 0;
    *out = c;
    return VLASOV_OK;
}

int vlasov_set_boundary(vlasov_ctx* c, int species, int side, int kind, const double* fluid5_dev) {
    if (!c || species < 0 || species >= c->ns || side < 0 || side > 1) return VLASOV_EINVAL;
    const int want = side == 0 ? c->G.bc_lo : c->G.bc_hi;
    if (kind != want) return VLASOV_EINVAL;
    if (kind == VLASOV_BC_FLUID && !fluid5_dev) return VLASOV_EINVAL;
    c->sp[species].fluid[side] = kind == VLASOV_BC_FLUID ? fluid5_dev : nullptr;
    return VLASOV_OK;
}

int vlasov_step(vlasov_ctx* c, double dt, const double* E_dev, const double* B_dev, uint32_t stages) {
    if (!c || !(dt == dt)) return VLASOV_EINVAL;
    const uint32_t vmask = c->order == VLASOV_ORDER_XVX ? VLASOV_STAGE_V : (VLASOV_STAGE_X1 | VLASOV_STAGE_X2);
    if ((stages & vmask) && (!E_dev || !B_dev)) return VLASOV_EINVAL;
    if (stages & ~(uint32_t)VLASOV_STAGE_ALL) return VLASOV_EINVAL;
    if (stages & VLASOV_STAGE_GHOST) {
        // a FLUID side needs its fluid state (vlasov_set_boundary) before the ghost fill can run
        for (int s = 0; s < c->ns; ++s) {
            if (c->G.bc_lo == VLASOV_BC_FLUID && !c->sp[s].fluid[0]) return VLASOV_EINVAL;
            if (c->G.bc_hi == VLASOV_BC_FLUID && !c->sp[s].fluid[1]) return VLASOV_EINVAL;
        }
    }
    if (stages & (VLASOV_STAGE_ALL & ~VLASOV_STAGE_MOMENTS)) c->mom_valid = 0;
    for (int s = 0; s < c->ns; ++s) {
        int e = species_step(c, s, dt, E_dev, B_dev, stages);
        if (e) return e;
    }
    if (stages & VLASOV_STAGE_MOMENTS) c->mom_valid = 1;
    return VLASOV_OK;
}

int vlasov_step_host(vlasov_ctx* c, double dt, const double* E_host, const double* B_host, uint32_t stages,
                     double* mom_host) {
    if (!c || !E_host || !B_host) return VLASOV_EINVAL;
    const size_t ncell = (size_t)c->G.nrows * c->G.nx;
    double* Ed = c->fields_stage;
    double* Bd = c->fields_stage + 3 * ncell;
    VL_CUDA_OK(cudaMemcpyAsync(Ed, E_host, 3 * ncell * 8, cudaMemcpyHostToDevice, c->stream));
    VL_CUDA_OK(cudaMemcpyAsync(Bd, B_host, 3 * ncell * 8, cudaMemcpyHostToDevice, c->stream));
    int e = vlasov_step(c, dt, Ed, Bd, stages);
    if (e) return e;
    if (mom_host) {
        e = ensure_moments(c);
        if (e) return e;
        for (int s = 0; s < c->ns; ++s)
            VL_CUDA_OK(cudaMemcpyAsync(mom_host + (size_t)s * 10 * ncell, c->mom + (size_t)s * 11 * ncell,
                                       10 * ncell * 8, cudaMemcpyDeviceToHost, c->stream));
    }
    return vlasov_check(c);
}

// One cycle of section 4.3 without the fluid step: currents -> fields half step ->
// Vlasov step with the new fields -> currents -> fields half step.
int vlasov_cycle(vlasov_ctx* c, double dt, int nsub, double* E_dev, double* B_dev) {
    if (!c || nsub <= 0 || !E_dev || !B_dev) return VLASOV_EINVAL;
    int e = ensure_moments(c); if (e) return e;
    e = launch_current(c, c->Jbuf); if (e) return e;
    e = launch_maxwell(c, dt / 2.0, nsub, E_dev, B_dev, c->Jbuf, c->Bavg); if (e) return e;
    e = vlasov_step(c, dt, E_dev, c->Bavg, VLASOV_STAGE_ALL); if (e) return e;
    e = launch_current(c, c->Jbuf); if (e) return e;
    return launch_maxwell(c, dt / 2.0, nsub, E_dev, B_dev, c->Jbuf, nullptr);
}

int vlasov_cycle_host(vlasov_ctx* c, double dt, int nsub, double* E_host, double* B_host, double* mom_host) {
    if (!c || !E_host || !B_host) return VLASOV_EINVAL;
    const size_t ncell = (size_t)c->G.nrows * c->G.nx;
    double* Ed = c->fields_stage;
    double* Bd = c->fields_stage + 3 * ncell;
    VL_CUDA_OK(cudaMemcpyAsync(Ed, E_host, 3 * ncell * 8, cudaMemcpyHostToDevice, c->stream));
    VL_CUDA_OK(cudaMemcpyAsync(Bd, B_host, 3 * ncell * 8, cudaMemcpyHostToDevice, c->stream));
    int e = vlasov_cycle(c, dt, nsub, Ed, Bd);
    if (e) return e;
    VL_CUDA_OK(cudaMemcpyAsync(E_host, Ed, 3 * ncell * 8, cudaMemcpyDeviceToHost, c->stream));
    VL_CUDA_OK(cudaMemcpyAsync(B_host, Bd, 3 * ncell * 8, cudaMemcpyDeviceToHost, c->stream));
    if (mom_host)
        for (int s = 0; s < c->ns; ++s)
            VL_CUDA_OK(cudaMemcpyAsync(mom_host + (size_t)s * 10 * ncell, c->mom + (size_t)s * 11 * ncell,
                                       10 * ncell * 8, cudaMemcpyDeviceToHost, c->stream));
    return vlasov_check(c);
}

// Per-kernel timing: event pairs around every launch while enabled (bench.py's roofline leg).
int vlasov_timing_enable(vlasov_ctx* c, int on) {
    if (!c) return VLASOV_EINVAL;
    if (on && !c->ev0) {
        c->ev0 = new (std::nothrow) cudaEvent_t[vlasov_ctx::MAX_REC];
        c->ev1 = new (std::nothrow) cudaEvent_t[vlasov_ctx::MAX_REC];
        c->rec_kind = new (std::nothrow) int[vlasov_ctx::MAX_REC];
        if (!c->ev0 || !c->ev1 || !c->rec_kind) return VLASOV_ECUDA;
        for (int i = 0; i < vlasov_ctx::MAX_REC; ++i) {
            VL_CUDA_OK(cudaEventCreate(&c->ev0[i]));
            VL_CUDA_OK(cudaEventCreate(&c->ev1[i]));
        }
    }
    c->timing = on ? 1 : 0;
    c->nrec = 0;
    return VLASOV_OK;
}

int vlasov_timing_read(vlasov_ctx* c, double* ms_by_kind, int64_t* count_by_kind, int nkinds) {
    if (!c || !ms_by_kind || !count_by_kind || nkinds < K_COUNT) return VLASOV_EINVAL;
    VL_CUDA_OK(cudaStreamSynchronize(c->stream));
    for (int k = 0; k < nkinds; ++k) { ms_by_kind[k] = 0.0; count_by_kind[k] = 0; }
    for (int i = 0; i < c->nrec; ++i) {
        float ms = 0.f;
        VL_CUDA_OK(cudaEventElapsedTime(&ms, c->ev0[i], c->ev1[i]));
        ms_by_kind[c->rec_kind[i]] += ms;
        count_by_kind[c->rec_kind[i]] += 1;
    }
    c->nrec = 0;
    return VLASOV_OK;
}

int vlasov_moments(vlasov_ctx* c, int species, double* mom_dev) {
    if (!c || species < 0 || species >= c->ns || !mom_dev) return VLASOV_EINVAL;
    if (((uintptr_t)mom_dev) & 7) return VLASOV_EALIGN;
    int e = ensure_moments(c);
    if (e) return e;
    const size_t ncell = (size_t)c->G.nrows * c->G.nx;
    VL_CUDA_OK(cudaMemcpyAsync(mom_dev, c->mom + (size_t)species * 11 * ncell, 10 * ncell * 8,
                               cudaMemcpyDeviceToDevice, c->stream));
    return VLASOV_OK;
}

// Section 4.1: the g interior rows next to border `side`, ghost-inclusive index of the first one
static inline int border_row0(const Geom& G, int side) { return side == 0 ? G.g : G.ny; }

// Moments (+ max) of the g interior rows next to border `side` of species s into dst [11][g*nx]: taken from the kept
// moments when the last step reduced them and f has not changed since, else reduced from f.  These launches exist only
// because a side is coupled: they carry the ghost timing kinds.
static int border_moments(vlasov_ctx* c, int s, int side, double* dst) {
    const long n = (long)c->G.g * c->G.nx, ncell = (long)c->G.nyg * c->G.nx;
    c->ghost_tag = 1;
    int e;
    if (c->mom_valid) e = launch_gather_rows(c, c->mom + (long)s * 11 * ncell, ncell, (long)border_row0(c->G, side) * c->G.nx, dst, n, 11);
    else e = launch_moments(c, c->sp[s], c->sp[s].f, dst, border_row0(c->G, side), c->G.g);
    c->ghost_tag = 0;
    return e;
}

int vlasov_fluid_boundary_mark(vlasov_ctx* c) {
    if (!c || c->G.g < 1 || c->G.ny < c->G.g || c->G.nz > 1) return VLASOV_EINVAL;
    const size_t n = (size_t)c->G.g * c->G.nx;
    for (int s = 0; s < c->ns; ++s)
        for (int side = 0; side < 2; ++side) {
            int e = border_moments(c, s, side, c->bmark + ((size_t)(s * 2 + side) * 11) * n);
            if (e) return e;
        }
    c->bmark_valid = 1;
    return VLASOV_OK;
}

int vlasov_fluid_boundary(vlasov_ctx* c, int species, int side, double theta, double* out_dev) {
    if (!c || species < 0 || species >= c->ns || side < 0 || side > 1 || !out_dev) return VLASOV_EINVAL;
    if (c->G.g < 1 || c->G.ny < c->G.g || !c->bmark_valid) return VLASOV_EINVAL;
    if (((uintptr_t)out_dev) & 7) return VLASOV_EALIGN;
    const size_t n = (size_t)c->G.g * c->G.nx;
    int e = border_moments(c, species, side, c->bcur);
    if (e) return e;
    c->ghost_tag = 1;
    e = launch_lerp(c, c->bmark + ((size_t)(species * 2 + side) * 11) * n, c->bcur, theta, out_dev, (long)(10 * n));
    c->ghost_tag = 0;
    return e;
}

int vlasov_current(vlasov_ctx* c, double* J_dev) {
    if (!c || !J_dev) return VLASOV_EINVAL;
    int e = ensure_moments(c);
    if (e) return e;
    return launch_current(c, J_dev);
}

int vlasov_maxwell(vlasov_ctx* c, double dt, int nsub, double* E_dev, double* B_dev, const double* J_dev,
                   double* Bavg_dev) {
    if (!c || nsub <= 0 || !E_dev || !B_dev || !J_dev) return VLASOV_EINVAL;
    return launch_maxwell(c, dt, nsub, E_dev, B_dev, J_dev, Bavg_dev);
}

int vlasov_set_option(vlasov_ctx* c, int option, int value) {
    if (!c) return VLASOV_EINVAL;
    if (option == VLASOV_OPT_FUSE_XY) { c->fuse_xy = value ? 1 : 0; return VLASOV_OK; }
    if (option == VLASOV_OPT_FUSE_MOMENTS) { c->fuse_mom = value ? 1 : 0; return VLASOV_OK; }
    return VLASOV_EINVAL;
}

int vlasov_touch(vlasov_ctx* c) {
    if (!c) return VLASOV_EINVAL;
    c->mom_valid = 0;
    return VLASOV_OK;
}

int vlasov_check(vlasov_ctx* c) {
    if (!c) return VLASOV_EINVAL;
    VL_CUDA_OK(cudaMemcpyAsync(c->h_err, c->errflag, sizeof(int), cudaMemcpyDeviceToHost, c->stream));
    VL_CUDA_OK(cudaStreamSynchronize(c->stream));
    const int e = *c->h_err;
    if (e) { VL_CUDA_OK(cudaMemsetAsync(c->errflag, 0, sizeof(int), c->stream)); }
    if (cudaGetLastError() != cudaSuccess) return VLASOV_ECUDA;
    return e;
}

int64_t vlasov_launch_count(const vlasov_ctx* c) { return c ? c->launches : 0; }

void vlasov_free(vlasov_ctx* c) {
    if (!c) return;
    if (c->h_err) cudaFreeHost(c->h_err);
    if (c->ev0) {
        for (int i = 0; i < vlasov_ctx::MAX_REC; ++i) { cudaEventDestroy(c->ev0[i]); cudaEventDestroy(c->ev1[i]); }
        delete[] c->ev0; delete[] c->ev1; delete[] c->rec_kind;
    }
    delete c;
}

const char* vlasov_strerror(int err) {
    switch (err) {
        case VLASOV_OK: return "ok";
        case VLASOV_EINVAL: return "invalid argument";
        case VLASOV_EALIGN: return "device pointer not 128-byte aligned";
        case VLASOV_ESHIFT: return "y shift reaches beyond the ghost rows";
        case VLASOV_EDOMAIN: return "Boris denominator or ghost-fill moment out of domain";
        case VLASOV_ECUDA: return "CUDA runtime error or no device";
        case VLASOV_ETOOBIG: return "fluid block larger than the static scratch array (VLASOV_FLUID_STATIC_SCRATCH_BYTES)";
        default: return "unknown error";
    }
}

}  // extern "C"
