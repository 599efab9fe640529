// Five-moment fluid step of the coupled scheme (section 3.2): CWENO3 in space, Shu-Osher SSP-RK3 in time,
// on the moment equations (5)-(7) PAPER.md:50-54 with the adiabatic closure (8) PAPER.md:61 and the Lorentz source, per
// species.  The paper gives the two names only; the details are reading R23 of DESIGN.md (Levy-Puppo-Russo weights,
// central-upwind flux at the face centre, dimension by dimension, sources from the stage's cell averages).
//
// The fluid grids of the paper's set-up are two-dimensional and tiny next to phase space ("negligible"),
// so the mapping is the plain one: one thread per (species, cell) and stage evaluates the four face fluxes of its cell
// from the 5 x 5 cross of cell averages around it (each face flux is evaluated by both neighbours with the same
// arithmetic: bit-identical, so the scheme conserves to round-off).  Three stage launches per step, ghost rows filled by
// a small kernel before each: periodic wrap, mirror image at a wall, or the caller's data at the stage time
// (section 4.1: "boundary conditions at times t, t + dt/2 and t + dt").
#include <cuda_runtime.h>
#include <stdint.h>
#include <atomic>
#include "../../include/vlasov.h"

namespace vlf {

constexpr int G = 2;                 // ghost rows per y side
constexpr double EPSW = 1e-6;        // epsilon of the nonlinear weights
constexpr double GAM = 5.0 / 3.0;    // eq. (8)

struct P {
    int nx, ny, ns;
    double dx, dy, dt;
    double qm[VLASOV_FLUID_MAX_SPECIES];
    int bc_lo, bc_hi;
};

// values of the CWENO3 reconstruction of cell averages (um, u, up) at the lower (w) and upper (e) face of the middle cell
__device__ __forceinline__ void cweno3(double um, double u, double up, double& w, double& e) {
    const double dl = u - um, dr = up - u, d2 = up - 2.0 * u + um, dc = up - um;
    const double il = dl * dl, ir = dr * dr, ic = (13.0 / 3.0) * d2 * d2 + 0.25 * dc * dc;
    const double tl = EPSW + il, tr = EPSW + ir, tc = EPSW + ic;
    const double al = 0.25 / (tl * tl), ar = 0.25 / (tr * tr), ac = 0.5 / (tc * tc);
    const double s = al + ar + ac;
    const double wl = al / s, wr = ar / s, wc = ac / s;
    e = wl * (u + 0.5 * dl) + wr * (u + 0.5 * dr) + wc * (u + d2 / 6.0 + 0.25 * dc);
    w = wl * (u - 0.5 * dl) + wr * (u - 0.5 * dr) + wc * (u + d2 / 6.0 - 0.25 * dc);
}

__device__ __forceinline__ double pressure(const double* U) {
    return (2.0 / 3.0) * U[4] - (1.0 / 3.0) * (U[1] * U[1] + U[2] * U[2] + U[3] * U[3]) / U[0];
}

// central-upwind flux through a face with normal direction d from the states Um (below the face) and Up (above)
__device__ __forceinline__ void face_flux(const double* Um, const double* Up, int d, double* H) {
    const double pm = pressure(Um), pp = pressure(Up);
    const double vm = Um[1 + d] / Um[0], vp = Up[1 + d] / Up[0];
    const double am = fabs(vm) + sqrt(GAM * pm / Um[0]), ap = fabs(vp) + sqrt(GAM * pp / Up[0]);
    const double a = fmax(am, ap);
    double Fm[5], Fp[5];
    Fm[0] = Um[1 + d]; Fp[0] = Up[1 + d];
    for (int k = 1; k < 4; ++k) { Fm[k] = Um[k] * vm; Fp[k] = Up[k] * vp; }
    Fm[1 + d] += pm; Fp[1 + d] += pp;
    Fm[4] = (Um[4] + pm) * vm; Fp[4] = (Up[4] + pp) * vp;
    for (int k = 0; k < 5; ++k) H[k] = 0.5 * (Fp[k] + Fm[k]) - 0.5 * a * (Up[k] - Um[k]);
}

// ghost rows of V [ns][5][ny+4][nx]; ghost_* [ns][5][2][nx] (this stage's), ascending y
__global__ void fluid_ghost_kernel(P p, double* __restrict__ V, const double* __restrict__ ghost_lo, const double* __restrict__ ghost_hi) {
    const int id = blockIdx.x * blockDim.x + threadIdx.x;
    const int n = p.ns * 5 * G * p.nx;
    if (id >= n) return;
    const int ix = id % p.nx, r = (id / p.nx) % G, k = (id / (p.nx * G)) % 5, s = id / (p.nx * G * 5);
    const int nyg = p.ny + 2 * G;
    double* Vk = V + ((long)(s * 5 + k) * nyg) * p.nx;
    {   // lower side: ghost row r
        double v;
        if (p.bc_lo == VLASOV_FLUID_BC_PERIODIC) v = Vk[(long)(p.ny + r) * p.nx + ix];
        else if (p.bc_lo == VLASOV_FLUID_BC_WALL) { v = Vk[(long)(2 * G - 1 - r) * p.nx + ix]; if (k == 2) v = -v; }
        else v = ghost_lo[((long)(s * 5 + k) * G + r) * p.nx + ix];
        Vk[(long)r * p.nx + ix] = v;
    }
    {   // upper side: ghost row ny + G + r
        double v;
        if (p.bc_hi == VLASOV_FLUID_BC_PERIODIC) v = Vk[(long)(G + r) * p.nx + ix];
        else if (p.bc_hi == VLASOV_FLUID_BC_WALL) { v = Vk[(long)(p.ny + G - 1 - r) * p.nx + ix]; if (k == 2) v = -v; }
        else v = ghost_hi[((long)(s * 5 + k) * G + r) * p.nx + ix];
        Vk[(long)(p.ny + G + r) * p.nx + ix] = v;
    }
}

// One Runge-Kutta stage: out = a0 U0 + b (V + dt L(V)) on the interior rows; V has its ghost rows filled.
__global__ void fluid_stage_kernel(P p, const double* U0, const double* __restrict__ V, double* out,
                                   const double* __restrict__ E, const double* __restrict__ B, double a0, double b) {
    const int id = blockIdx.x * blockDim.x + threadIdx.x;
    const int ncell = p.nx * p.ny;
    if (id >= ncell * p.ns) return;
    const int s = id / ncell, c = id - s * ncell;
    const int j = G + c / p.nx, i = c % p.nx;
    const int nyg = p.ny + 2 * G;
    const long PL = (long)nyg * p.nx;
    const double* Vs = V + (long)s * 5 * PL;
    auto at = [&](int k, int jj, int ii) { return Vs[k * PL + (long)jj * p.nx + ii]; };
    auto wrap = [&](int ii) { return ii < 0 ? ii + p.nx : (ii >= p.nx ? ii - p.nx : ii); };
    double L[5] = {0, 0, 0, 0, 0};
    for (int d = 0; d < 2; ++d) {
        // reconstructions of the cells -1, 0, +1 along d: lower and upper face values of each
        double lo[3][5], hi[3][5];
        for (int k = 0; k < 5; ++k) {
            double q[5];
            for (int o = -2; o <= 2; ++o) q[o + 2] = d == 0 ? at(k, j, wrap(i + o)) : at(k, j + o, i);
            for (int cc = 0; cc < 3; ++cc) cweno3(q[cc], q[cc + 1], q[cc + 2], lo[cc][k], hi[cc][k]);
        }
        double Hm[5], Hp[5];
        face_flux(hi[0], lo[1], d, Hm);        // face between cell -1 and cell 0
        face_flux(hi[1], lo[2], d, Hp);        // face between cell 0 and cell +1
        const double h = d == 0 ? p.dx : p.dy;
        for (int k = 0; k < 5; ++k) L[k] -= (Hp[k] - Hm[k]) / h;
    }
    // Lorentz source, eqs. (6), (7): (q/m)(rho E + u x B), (q/m) u . E, fields at the cell centre
    const long cc = (long)j * p.nx + i;
    const double rho = at(0, j, i), ux = at(1, j, i), uy = at(2, j, i), uz = at(3, j, i), en = at(4, j, i);
    const double Ex = E[cc], Ey = E[PL + cc], Ez = E[2 * PL + cc], Bx = B[cc], By = B[PL + cc], Bz = B[2 * PL + cc];
    const double qm = p.qm[s];
    L[1] += qm * (rho * Ex + (uy * Bz - uz * By));
    L[2] += qm * (rho * Ey + (uz * Bx - ux * Bz));
    L[3] += qm * (rho * Ez + (ux * By - uy * Bx));
    L[4] += qm * (ux * Ex + uy * Ey + uz * Ez);
    const double v[5] = {rho, ux, uy, uz, en};
    for (int k = 0; k < 5; ++k) {
        const long o = ((long)s * 5 + k) * PL + cc;
        out[o] = a0 * U0[o] + b * (v[k] + p.dt * L[k]);
    }
}

__global__ void from_moments_kernel(const double* __restrict__ mom, double m, double* __restrict__ U, long n) {
    const long i = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    U[i] = m * mom[i];
    U[n + i] = m * mom[n + i];
    U[2 * n + i] = m * mom[2 * n + i];
    U[3 * n + i] = m * mom[3 * n + i];
    U[4 * n + i] = 0.5 * m * (mom[4 * n + i] + mom[5 * n + i] + mom[6 * n + i]);
}

__global__ void to_boundary_kernel(const double* __restrict__ U, double m, double* __restrict__ b5, long n) {
    const long i = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const double v[5] = {U[i], U[n + i], U[2 * n + i], U[3 * n + i], U[4 * n + i]};
    b5[i] = v[0] / m;
    b5[n + i] = v[1] / v[0];
    b5[2 * n + i] = v[2] / v[0];
    b5[3 * n + i] = v[3] / v[0];
    b5[4 * n + i] = pressure(v);
}

}  // namespace vlf

extern "C" {

size_t vlasov_fluid_scratch_bytes(const vlasov_fluid_config* cfg) {
    if (!cfg || cfg->nx < 1 || cfg->ny < 1 || cfg->nspecies < 1 || cfg->nspecies > VLASOV_FLUID_MAX_SPECIES) return 0;
    return 2 * (size_t)cfg->nspecies * 5 * (cfg->ny + 2 * vlf::G) * cfg->nx * sizeof(double);
}

int vlasov_fluid_step(const vlasov_fluid_config* cfg, double dt, double* U_dev, const double* E_dev, const double* B_dev,
                      const double* ghost_lo_dev, const double* ghost_hi_dev, void* scratch_dev, size_t scratch_bytes) {
    const size_t need = vlasov_fluid_scratch_bytes(cfg);
    if (!need || !U_dev || !E_dev || !B_dev || !scratch_dev || scratch_bytes < need || !(dt == dt)) return VLASOV_EINVAL;
    if (!(cfg->dx > 0.0) || !(cfg->dy > 0.0)) return VLASOV_EINVAL;
    if (cfg->bc_y_lo < 0 || cfg->bc_y_lo > 2 || cfg->bc_y_hi < 0 || cfg->bc_y_hi > 2) return VLASOV_EINVAL;
    if ((cfg->bc_y_lo == VLASOV_FLUID_BC_PERIODIC) != (cfg->bc_y_hi == VLASOV_FLUID_BC_PERIODIC)) return VLASOV_EINVAL;
    if ((cfg->bc_y_lo == VLASOV_FLUID_BC_COUPLED && !ghost_lo_dev) || (cfg->bc_y_hi == VLASOV_FLUID_BC_COUPLED && !ghost_hi_dev)) return VLASOV_EINVAL;
    if (cfg->bc_y_lo != VLASOV_FLUID_BC_COUPLED && cfg->ny < vlf::G) return VLASOV_EINVAL;
    if ((((uintptr_t)U_dev) | ((uintptr_t)scratch_dev)) & 7) return VLASOV_EALIGN;
    vlf::P p;
    p.nx = cfg->nx; p.ny = cfg->ny; p.ns = cfg->nspecies; p.dx = cfg->dx; p.dy = cfg->dy; p.dt = dt;
    for (int s = 0; s < p.ns; ++s) {
        if (!(cfg->m[s] > 0.0)) return VLASOV_EINVAL;
        p.qm[s] = cfg->q[s] / cfg->m[s];
    }
    p.bc_lo = cfg->bc_y_lo; p.bc_hi = cfg->bc_y_hi;
    cudaStream_t st = (cudaStream_t)cfg->stream;
    const size_t n = need / 2 / sizeof(double);
    double* U1 = (double*)scratch_dev;
    double* U2 = U1 + n;
    const size_t gstage = (size_t)p.ns * 5 * vlf::G * p.nx;     // ghost data of one stage
    const int ng = p.ns * 5 * vlf::G * p.nx, nc = p.ns * p.nx * p.ny;
    auto ghosts = [&](double* V, int stage) {
        vlf::fluid_ghost_kernel<<<(ng + 127) / 128, 128, 0, st>>>(p, V, ghost_lo_dev ? ghost_lo_dev + stage * gstage : nullptr,
                                                               ghost_hi_dev ? ghost_hi_dev + stage * gstage : nullptr);
    };
    // Shu-Osher SSP-RK3: stages at t, t + dt, t + dt/2
    ghosts(U_dev, 0);
    vlf::fluid_stage_kernel<<<(nc + 127) / 128, 128, 0, st>>>(p, U_dev, U_dev, U1, E_dev, B_dev, 0.0, 1.0);
    ghosts(U1, 1);
    vlf::fluid_stage_kernel<<<(nc + 127) / 128, 128, 0, st>>>(p, U_dev, U1, U2, E_dev, B_dev, 0.75, 0.25);
    ghosts(U2, 2);
    // the last stage reads U0 = U_dev only at the cell it writes: in place is safe
    vlf::fluid_stage_kernel<<<(nc + 127) / 128, 128, 0, st>>>(p, U_dev, U2, U_dev, E_dev, B_dev, 1.0 / 3.0, 2.0 / 3.0);
    return cudaGetLastError() == cudaSuccess ? VLASOV_OK : VLASOV_ECUDA;
}

int vlasov_fluid_from_moments(const double* mom10_dev, double m, double* U5_dev, long n, void* stream) {
    if (!mom10_dev || !U5_dev || n <= 0 || !(m > 0.0)) return VLASOV_EINVAL;
    vlf::from_moments_kernel<<<(unsigned)((n + 127) / 128), 128, 0, (cudaStream_t)stream>>>(mom10_dev, m, U5_dev, n);
    return cudaGetLastError() == cudaSuccess ? VLASOV_OK : VLASOV_ECUDA;
}

int vlasov_fluid_to_boundary(const double* U5_dev, double m, double* fluid5_dev, long n, void* stream) {
    if (!U5_dev || !fluid5_dev || n <= 0 || !(m > 0.0)) return VLASOV_EINVAL;
    vlf::to_boundary_kernel<<<(unsigned)((n + 127) / 128), 128, 0, (cudaStream_t)stream>>>(U5_dev, m, fluid5_dev, n);
    return cudaGetLastError() == cudaSuccess ? VLASOV_OK : VLASOV_ECUDA;
}

}  // extern "C"

// ---- vlasov_fluid_step without an allocation anywhere (include/vlasov.h) ---------------------------------------------
// The two stage buffers live in the library image.  In host code `fluid_static_scratch` is a host-side stand-in, not a
// device address: the address a kernel may use comes from cudaGetSymbolAddress, once per device, with that device current.
static __device__ __align__(256) unsigned char fluid_static_scratch[VLASOV_FLUID_STATIC_SCRATCH_BYTES];

namespace vlf {

constexpr int MAX_DEVICES = 64;
std::atomic<void*> static_scratch_addr[MAX_DEVICES];      // zero-initialised; one slot per device ordinal

// device address of fluid_static_scratch on the current device (nullptr on a CUDA error)
static void* static_scratch_of_current_device() {
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= MAX_DEVICES) return nullptr;
    void* p = static_scratch_addr[dev].load(std::memory_order_acquire);
    if (p) return p;
    if (cudaGetSymbolAddress(&p, fluid_static_scratch) != cudaSuccess || !p) return nullptr;
    static_scratch_addr[dev].store(p, std::memory_order_release);     // same value whoever gets here first
    return p;
}

}  // namespace vlf

extern "C" int vlasov_fluid_step_static(const vlasov_fluid_config* cfg, double dt, double* U_dev, const double* E_dev,
                                        const double* B_dev, const double* ghost_lo_dev, const double* ghost_hi_dev) {
    const size_t need = vlasov_fluid_scratch_bytes(cfg);
    if (!need) return VLASOV_EINVAL;
    if (need > (size_t)VLASOV_FLUID_STATIC_SCRATCH_BYTES) return VLASOV_ETOOBIG;
    void* scratch = vlf::static_scratch_of_current_device();
    if (!scratch) return VLASOV_ECUDA;
    return vlasov_fluid_step(cfg, dt, U_dev, E_dev, B_dev, ghost_lo_dev, ghost_hi_dev, scratch, need);
}
