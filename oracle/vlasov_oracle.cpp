// ORACLE -- TEST INFRASTRUCTURE ONLY.
//
// Plain fp64 CPU implementation of the Vlasov full-step hot path of arXiv 1406.5445
// (Rieke, Trost, Grauer), written from the paper step by step in the paper's order
// and notation.  It shares no code, header, table or helper with the CUDA path under
// paper_1406_5445_b200/csrc/.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
// --impl reference legs may load it.  It is never tuned; OpenMP only spreads independent
// phase-space lines / spatial cells over the host cores.
//
// Layout (same as the library's, because it is the interface):
//   f[iy_g][ix][ivx][ivy][ivz], iy_g = 0..ny+2g-1 (g ghost rows per y side), fp64.
//   fields  E,B,J : [3][ny_g][nx];  moments: [10][ny_g][nx].
//
// Pins (tests/test_oracle_*.py): T1..T17 of DESIGN.md, the VXV pins (orc_step with order = 1: T10/T11/T5/T16 under
// that order, Landau rate under VXV), the PEC-row pins of orc_field_at_cell and orc_current, and -- for the cycle
// composed from these functions in oracle.py -- C1, C2; the 3D3V functions at the end of this file: D1..D6
// (tests/test_oracle_3d.py).  Every function here is pinned.  Readings the paper leaves
// open and for which no outside fact exists are DECLARED DEFINITIONS: limiter under compressive
// velocity shifts (R6/R15d), zeroth-order ghost extrapolation (R15a), isotropic target temperature (R15c), ghost-row
// Dirichlet reuse (R16), the choice of Yee positions (R17).
//
// Build: g++ -O2 -ffp-contract=off -fopenmp -shared -fPIC vlasov_oracle.cpp -o liboracle.so

#include <cmath>
#include <cstdint>
#include <cstring>
#include <vector>
#include <algorithm>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

enum { BC_PERIODIC = 0, BC_REFLECT = 1, BC_FLUID = 2 };
enum { ERR_OK = 0, ERR_SHIFT = -3, ERR_DOMAIN = -4 };

// ---------------------------------------------------------------------------------------------
// PFC slope limiters, eqs. (43), (44).  Reading R6: equal neighbours -> eps=1,
// result clamped to [0,1].  limiter==0 -> eps=1 (unlimited third-order scheme).
// ---------------------------------------------------------------------------------------------
inline double clamp01(double e) { return e < 0.0 ? 0.0 : (e > 1.0 ? 1.0 : e); }

inline double eps_plus(double fj, double fjp1, double finf, int limiter) {
    if (!limiter) return 1.0;
    double d = fjp1 - fj;
    double e = 1.0;
    if (d > 0.0)      e = std::min(1.0, 2.0 * fj / d);
    else if (d < 0.0) e = std::min(1.0, -2.0 * (finf - fj) / d);
    return clamp01(e);
}

inline double eps_minus(double fjm1, double fj, double finf, int limiter) {
    if (!limiter) return 1.0;
    double d = fj - fjm1;
    double e = 1.0;
    if (d > 0.0)      e = std::min(1.0, 2.0 * (finf - fj) / d);
    else if (d < 0.0) e = std::min(1.0, -2.0 * fj / d);
    return clamp01(e);
}

// ---------------------------------------------------------------------------------------------
// Flux through face i+1/2, eq. (46) for sigma >= 0 and eq. (47) for sigma < 0 (
// eq. 47's whole-cell sum repaired to -sum_{k=i+1}^{j-1}, reading R5).  sigma is the signed
// distance, in cells, from the face back to the foot of the characteristic.  get(k) returns the
// cell average f_k for ANY integer k (the boundary condition lives in get).
// ---------------------------------------------------------------------------------------------
template <class Get>
inline double pfc_flux(Get get, long i, double sigma, double finf, int limiter) {
    if (sigma >= 0.0) {
        double nf = std::floor(sigma);
        long n = (long)nf;
        double a = sigma - nf;          // alpha in [0,1)
        long j = i - n;
        double sum = 0.0;
        for (long k = j + 1; k <= i; ++k) sum += get(k);
        double fjm = get(j - 1), fj = get(j), fjp = get(j + 1);
        double ep = eps_plus(fj, fjp, finf, limiter);
        double em = eps_minus(fjm, fj, finf, limiter);
        return sum + a * (fj + (ep / 6.0) * (1.0 - a) * (2.0 - a) * (fjp - fj)
                             + (em / 6.0) * (1.0 - a) * (1.0 + a) * (fj - fjm));
    } else {
        double s = -sigma;
        double nf = std::floor(s);
        long n = (long)nf;
        double a = -(s - nf);           // alpha in (-1,0]
        long j = i + 1 + n;
        double sum = 0.0;
        for (long k = i + 1; k <= j - 1; ++k) sum += get(k);
        double fjm = get(j - 1), fj = get(j), fjp = get(j + 1);
        double ep = eps_plus(fj, fjp, finf, limiter);
        double em = eps_minus(fjm, fj, finf, limiter);
        return -sum + a * (fj - (ep / 6.0) * (1.0 - a) * (1.0 + a) * (fjp - fj)
                              - (em / 6.0) * (2.0 + a) * (1.0 + a) * (fj - fjm));
    }
}

// ---------------------------------------------------------------------------------------------
// 1D conservative remap of one line, eq. (38): f'_i = f_i + (Phi_{i-1/2} - Phi_{i+1/2}),
// all fluxes from the OLD f.  sigma[k], k=0..n, is the shift of face k-1/2 (face k lies between
// cells k-1 and k).  bc: 0 periodic, 1 zero outside and zero flux through the two outer faces (R7).
// ---------------------------------------------------------------------------------------------
void remap_line(const double* f, long n, const double* sigma, int bc, double finf, int limiter,
                double* out) {
    std::vector<double> phi(n + 1);
    if (bc == 0) {
        auto get = [&](long k) { long m = k % n; if (m < 0) m += n; return f[m]; };
        for (long k = 0; k <= n; ++k) phi[k] = pfc_flux(get, k - 1, sigma[k], finf, limiter);
    } else {
        auto get = [&](long k) { return (k < 0 || k >= n) ? 0.0 : f[k]; };
        phi[0] = 0.0; phi[n] = 0.0;
        for (long k = 1; k < n; ++k) phi[k] = pfc_flux(get, k - 1, sigma[k], finf, limiter);
    }
    for (long i = 0; i < n; ++i) out[i] = f[i] + (phi[i] - phi[i + 1]);
}

struct Grid {
    int nx, ny, g, nyg;
    int nv[3];
    long nvtot;
    double vmin[3], dv[3];
};

inline double vcen(const Grid& G, int d, int k) { return G.vmin[d] + (k + 0.5) * G.dv[d]; }
inline double vface(const Grid& G, int d, int k) { return G.vmin[d] + k * G.dv[d]; }

Grid make_grid(int nx, int ny, int g, const int* nv, const double* vmin, const double* vmax) {
    Grid G;
    G.nx = nx; G.ny = ny; G.g = g; G.nyg = ny + 2 * g;
    G.nvtot = 1;
    for (int d = 0; d < 3; ++d) {
        G.nv[d] = nv[d]; G.vmin[d] = vmin[d];
        G.dv[d] = (vmax[d] - vmin[d]) / nv[d];
        G.nvtot *= nv[d];
    }
    return G;
}

}  // namespace

extern "C" {

// --- 8(c)-1: the core routine, exported for the pins ------------------------------------------
void orc_remap1d(const double* f, long n, const double* sigma, int bc, double finf, int limiter,
                 double* out) {
    remap_line(f, n, sigma, bc, finf, limiter, out);
}

// --- a1/a8: x half-sweep T(dts * v_x d/dx), periodic, all rows incl. ghost rows ----------------
// sigma = v_x[ivx] * dts / dx on every face (eqs. 38, 46/47).
void orc_sweep_x(double* f, int nx, int ny, int g, const int* nv, const double* vmin,
                 const double* vmax, double dx, double dts, double finf, int limiter) {
    Grid G = make_grid(nx, ny, g, nv, vmin, vmax);
    const long S = G.nvtot;  // stride between x neighbours
#pragma omp parallel
    {
        std::vector<double> line(nx), out(nx), sig(nx + 1);
#pragma omp for collapse(2) schedule(static)
        for (int iy = 0; iy < G.nyg; ++iy)
            for (long v = 0; v < S; ++v) {
                int ivx = (int)(v / ((long)nv[1] * nv[2]));
                double s = vcen(G, 0, ivx) * dts / dx;
                for (int k = 0; k <= nx; ++k) sig[k] = s;
                double* base = f + ((long)iy * nx) * S + v;
                for (int i = 0; i < nx; ++i) line[i] = base[(long)i * S];
                remap_line(line.data(), nx, sig.data(), 0, finf, limiter, out.data());
                for (int i = 0; i < nx; ++i) base[(long)i * S] = out[i];
            }
    }
}

// --- a2/a7: y half-sweep.  Interior rows only are updated; rows outside [0,ny) are supplied by the
// boundary kind of that side: PERIODIC wrap, REFLECT (R19: f(y_w+eta,vx,vy,vz)=f(y_w-eta,vx,-vy,vz),
// needs a symmetric v_y grid), FLUID (ghost rows, Dirichlet data, R16).  Returns ERR_SHIFT when a
// FLUID side is asked for a row beyond its ghost rows (R9).
int orc_sweep_y(double* f, int nx, int ny, int g, const int* nv, const double* vmin,
                const double* vmax, double dy, double dts, double finf, int limiter, int bc_lo,
                int bc_hi) {
    Grid G = make_grid(nx, ny, g, nv, vmin, vmax);
    const long S = G.nvtot;
    const long rowstride = (long)nx * S;
    int err = ERR_OK;
    // eq. (38): every flux is taken from the OLD f.  A REFLECT side reads the line with v_y mirrored, which
    // is another line of the same array, so the sweep reads from a snapshot and writes into f.
    const std::vector<double> old(f, f + (long)G.nyg * rowstride);
#pragma omp parallel
    {
        std::vector<double> out(ny), sig(ny + 1);
#pragma omp for collapse(2) schedule(static)
        for (int ix = 0; ix < nx; ++ix)
            for (long v = 0; v < S; ++v) {
                int ivy = (int)((v / nv[2]) % nv[1]);
                long vmir = v + (long)(nv[1] - 1 - 2 * ivy) * nv[2];  // same cell with ivy mirrored
                double s = vcen(G, 1, ivy) * dts / dy;
                int lerr = ERR_OK;
                auto get = [&](long r) -> double {
                    long vv = v;
                    for (int guard = 0; guard < 4 && (r < 0 || r >= ny); ++guard) {
                        if (r < 0) {
                            if (bc_lo == BC_PERIODIC) r += ny;
                            else if (bc_lo == BC_REFLECT) { r = -1 - r; vv = (vv == v) ? vmir : v; }
                            else { if (r + g < 0) { lerr = ERR_SHIFT; return 0.0; }
                                   return old[(r + g) * rowstride + (long)ix * S + vv]; }
                        } else {
                            if (bc_hi == BC_PERIODIC) r -= ny;
                            else if (bc_hi == BC_REFLECT) { r = 2L * ny - 1 - r; vv = (vv == v) ? vmir : v; }
                            else { if (r + g >= G.nyg) { lerr = ERR_SHIFT; return 0.0; }
                                   return old[(r + g) * rowstride + (long)ix * S + vv]; }
                        }
                    }
                    if (r < 0 || r >= ny) { lerr = ERR_SHIFT; return 0.0; }
                    return old[(r + g) * rowstride + (long)ix * S + vv];
                };
                std::vector<double> phi(ny + 1);
                for (int k = 0; k <= ny; ++k) phi[k] = pfc_flux(get, k - 1, s, finf, limiter);
                for (int i = 0; i < ny; ++i) out[i] = get(i) + (phi[i] - phi[i + 1]);
                for (int i = 0; i < ny; ++i) f[(long)(i + g) * rowstride + (long)ix * S + v] = out[i];
                if (lerr) {
#pragma omp critical
                    err = lerr;
                }
            }
    }
    return err;
}

// --- a3: fields at the centre of spatial cell (ix, j) (j = ghost-inclusive row) ----------------
// fields_yee == 0: arrays are cell-centred.  fields_yee == 1: 2D Yee positions of reading R17,
// cell (i,j) spans [i dx,(i+1)dx] x [j dy,(j+1)dy]:  Ex(i+1/2,j) Ey(i,j+1/2) Ez(i,j)
// Bx(i,j+1/2) By(i+1/2,j) Bz(i+1/2,j+1/2); linear interpolation to the centre.
// Row j+1 beyond the array: periodic wrap if wall==0, PEC wall value 0 if wall==1.
void orc_field_at_cell(const double* E, const double* B, int nx, int nyg, int fields_yee, int wall,
                       int ix, int j, double* Ec, double* Bc) {
    const long P = (long)nyg * nx;
    if (!fields_yee) {
        for (int d = 0; d < 3; ++d) { Ec[d] = E[d * P + (long)j * nx + ix]; Bc[d] = B[d * P + (long)j * nx + ix]; }
        return;
    }
    int ip = (ix + 1) % nx;
    int jp = j + 1;
    double up = 1.0;   // weight of row j+1 values that vanish on a PEC wall
    if (jp >= nyg) { jp = 0; if (wall) up = 0.0; }
    auto at = [&](const double* A, int d, int jj, int ii) { return A[d * P + (long)jj * nx + ii]; };
    Ec[0] = 0.5 * (at(E, 0, j, ix) + up * at(E, 0, jp, ix));
    Ec[1] = 0.5 * (at(E, 1, j, ix) + at(E, 1, j, ip));
    Ec[2] = 0.25 * (at(E, 2, j, ix) + at(E, 2, j, ip) + up * at(E, 2, jp, ix) + up * at(E, 2, jp, ip));
    Bc[0] = 0.5 * (at(B, 0, j, ix) + at(B, 0, j, ip));
    Bc[1] = 0.5 * (at(B, 1, j, ix) + up * at(B, 1, jp, ix));
    Bc[2] = at(B, 2, j, ix);
}

// --- feet of the three velocity sweeps, eqs. (35), (34), (33) with the half-kicks of eq. (26) ---
// (reading R10).  dir = 0: vx sweep, face a, transverse centres (vy, vz) read as v^n.
//                 dir = 1: vy sweep, face b, vx read as v^{n+1}, vz as v^n.
//                 dir = 2: vz sweep, face c, vx, vy read as v^{n+1}.
// Returns the foot in v^n coordinates.  t, s of eq. (28); h = (q/m)(dt/2)E.
double orc_vfoot(int dir, double face, double w1, double w2, const double* t, const double* s,
                 const double* h) {
    const double tx = t[0], ty = t[1], tz = t[2], sx = s[0], sy = s[1], sz = s[2];
    if (dir == 0) {
        double vxp = face - h[0], vym = w1 + h[1], vzm = w2 + h[2];
        double D1 = 1.0 - ty * sy - tz * sz;
        double vxm = (vxp - vym * (tx * sy + sz) - vzm * (tx * sz - sy)) / D1;          // eq. (35)
        return vxm - h[0];
    } else if (dir == 1) {
        double vxp = w1 - h[0], vyp = face - h[1], vzm = w2 + h[2];
        double D2 = 1.0 - tx * sx - ty * sy;
        double g = (ty * sz - sx) / D2;
        double vym = vxp * (sx * ty + sz - (tz * sx - sy) * g)
                   + vyp * (1.0 - tx * sx - tz * sz - (tz * sy + sx) * g) + vzm * g;     // eq. (34)
        return vym - h[1];
    } else {
        double vxp = w1 - h[0], vyp = w2 - h[1], vzp = face - h[2];
        double vzm = vxp * (tz * sx - sy) + vyp * (tz * sy + sx) + vzp * (1.0 - tx * sx - ty * sy);  // eq. (33)
        return vzm - h[2];
    }
}

// Backward Boris push, eqs. (31), (32) with (26): v^n from v^{n+1}.  Exported for pins T8/T9 only
// (the sweeps use orc_vfoot).
void orc_boris_back(const double* vnp1, const double* t, const double* s, const double* h, double* vn) {
    double vp[3] = {vnp1[0] - h[0], vnp1[1] - h[1], vnp1[2] - h[2]};
    double w[3] = {vp[0] - (vp[1] * t[2] - vp[2] * t[1]),
                   vp[1] - (vp[2] * t[0] - vp[0] * t[2]),
                   vp[2] - (vp[0] * t[1] - vp[1] * t[0])};                      // eq. (31)
    double vm[3] = {vp[0] - (w[1] * s[2] - w[2] * s[1]),
                    vp[1] - (w[2] * s[0] - w[0] * s[2]),
                    vp[2] - (w[0] * s[1] - w[1] * s[0])};                       // eq. (32)
    for (int d = 0; d < 3; ++d) vn[d] = vm[d] - h[d];
}

// t, s, h of eqs. (26), (28) from the cell-centre fields.  Returns ERR_DOMAIN when a denominator
// of eqs. (34)/(35) is not positive (R13).
int orc_boris_coeffs(const double* Ec, const double* Bc, double q, double m, double dt, double* t,
                     double* s, double* h) {
    double qm = q / m;
    double t2 = 0.0;
    for (int d = 0; d < 3; ++d) { t[d] = qm * (dt / 2.0) * Bc[d]; h[d] = qm * (dt / 2.0) * Ec[d]; t2 += t[d] * t[d]; }
    for (int d = 0; d < 3; ++d) s[d] = 2.0 * t[d] / (1.0 + t2);
    double D1 = 1.0 - t[1] * s[1] - t[2] * s[2];
    double D2 = 1.0 - t[0] * s[0] - t[1] * s[1];
    return (D1 > 0.0 && D2 > 0.0) ? ERR_OK : ERR_DOMAIN;
}

// --- a4..a6 on ONE velocity block fb[ivx][ivy][ivz] (in place), order vx -> vy -> vz ------------
// (PAPER.md:229).  order_reversed != 0 applies vz -> vy -> vx instead (pin T9's negative control).
void orc_vsweeps_block(double* fb, const int* nv, const double* vmin, const double* vmax,
                       const double* t, const double* s, const double* h, double finf, int limiter,
                       int order_reversed) {
    int nvv[3] = {nv[0], nv[1], nv[2]};
    Grid G = make_grid(1, 1, 0, nvv, vmin, vmax);
    const long st[3] = {(long)nv[1] * nv[2], (long)nv[2], 1};
    const int maxn = std::max(nv[0], std::max(nv[1], nv[2]));
    std::vector<double> line(maxn), out(maxn), sig(maxn + 1);
    for (int step = 0; step < 3; ++step) {
        int d = order_reversed ? 2 - step : step;
        int d1 = (d == 0) ? 1 : 0;          // first transverse direction (lower axis index)
        int d2 = (d == 2) ? 1 : 2;          // second transverse direction
        for (int k1 = 0; k1 < nv[d1]; ++k1)
            for (int k2 = 0; k2 < nv[d2]; ++k2) {
                double w1 = vcen(G, d1, k1), w2 = vcen(G, d2, k2);
                double* base = fb + k1 * st[d1] + k2 * st[d2];
                int n = nv[d];
                for (int k = 0; k <= n; ++k) {
                    double face = vface(G, d, k);
                    double foot = orc_vfoot(d, face, w1, w2, t, s, h);
                    sig[k] = (face - foot) / G.dv[d];
                }
                for (int k = 0; k < n; ++k) line[k] = base[k * st[d]];
                remap_line(line.data(), n, sig.data(), 1, finf, limiter, out.data());
                for (int k = 0; k < n; ++k) base[k * st[d]] = out[k];
            }
    }
}

// --- a3..a6 for every spatial cell, ghost rows included (R16) ---------------------------------
int orc_vstep(double* f, int nx, int ny, int g, const int* nv, const double* vmin, const double* vmax,
              double q, double m, double dt, const double* E, const double* B, int fields_yee,
              int wall, double finf, int limiter) {
    Grid G = make_grid(nx, ny, g, nv, vmin, vmax);
    int err = ERR_OK;
#pragma omp parallel for collapse(2) schedule(static)
    for (int j = 0; j < G.nyg; ++j)
        for (int ix = 0; ix < nx; ++ix) {
            double Ec[3], Bc[3], t[3], s[3], h[3];
            orc_field_at_cell(E, B, nx, G.nyg, fields_yee, wall, ix, j, Ec, Bc);
            int e = orc_boris_coeffs(Ec, Bc, q, m, dt, t, s, h);
            if (e) {
#pragma omp critical
                err = e;
                continue;
            }
            orc_vsweeps_block(f + ((long)j * nx + ix) * G.nvtot, nv, vmin, vmax, t, s, h, finf, limiter, 0);
        }
    return err;
}

// --- a9: raw velocity moments of one block, eqs. (2)-(4) as midpoint sums (8(c)-3) -------------
// out[10] = M0, M1x, M1y, M1z, M2xx, M2yy, M2zz, M2xy, M2xz, M2yz, each times dvx*dvy*dvz.
void orc_moments_block(const double* fb, const int* nv, const double* vmin, const double* vmax,
                       double* out) {
    int nvv[3] = {nv[0], nv[1], nv[2]};
    Grid G = make_grid(1, 1, 0, nvv, vmin, vmax);
    double M[10] = {0, 0, 0, 0, 0, 0, 0, 0, 0, 0};
    for (int a = 0; a < nv[0]; ++a)
        for (int b = 0; b < nv[1]; ++b)
            for (int c = 0; c < nv[2]; ++c) {
                double fv = fb[((long)a * nv[1] + b) * nv[2] + c];
                double vx = vcen(G, 0, a), vy = vcen(G, 1, b), vz = vcen(G, 2, c);
                M[0] += fv;
                M[1] += vx * fv; M[2] += vy * fv; M[3] += vz * fv;
                M[4] += vx * vx * fv; M[5] += vy * vy * fv; M[6] += vz * vz * fv;
                M[7] += vx * vy * fv; M[8] += vx * vz * fv; M[9] += vy * vz * fv;
            }
    double dv3 = G.dv[0] * G.dv[1] * G.dv[2];
    for (int k = 0; k < 10; ++k) out[k] = M[k] * dv3;
}

void orc_moments(const double* f, int nx, int ny, int g, const int* nv, const double* vmin,
                 const double* vmax, double* mom /*[10][nyg][nx]*/) {
    Grid G = make_grid(nx, ny, g, nv, vmin, vmax);
    const long P = (long)G.nyg * nx;
#pragma omp parallel for schedule(static)
    for (long c = 0; c < P; ++c) {
        double M[10];
        orc_moments_block(f + c * G.nvtot, nv, vmin, vmax, M);
        for (int k = 0; k < 10; ++k) mom[k * P + c] = M[k];
    }
}

// --- a0: ghost fill for one y side of kind FLUID, 8(c)-4 (eqs. 48-50, 63) ----
// fluid5: [5][g][nx] = n, ux, uy, uz (bulk velocity), p (scalar pressure) of each ghost cell,
// layer index l = 0..g-1 counted OUTWARD from the kinetic edge.
int orc_ghost_fill(double* f, int nx, int ny, int g, const int* nv, const double* vmin,
                   const double* vmax, double m, int side, const double* fluid5, int limiter) {
    Grid G = make_grid(nx, ny, g, nv, vmin, vmax);
    const long S = G.nvtot;
    int err = ERR_OK;
    const int edge_row = side == 0 ? g : g + ny - 1;
#pragma omp parallel for collapse(2) schedule(static)
    for (int l = 0; l < g; ++l)
        for (int ix = 0; ix < nx; ++ix) {
            const int row = side == 0 ? g - 1 - l : g + ny + l;
            const double* fe = f + ((long)edge_row * nx + ix) * S;     // f^E: zeroth-order extrapolation (R15a)
            double* fm = f + ((long)row * nx + ix) * S;
            double M[10];
            orc_moments_block(fe, nv, vmin, vmax, M);                    // step 2, eq. (48) per direction
            double nE = M[0];
            double nM = fluid5[(0L * g + l) * nx + ix];
            double VM[3] = {fluid5[(1L * g + l) * nx + ix], fluid5[(2L * g + l) * nx + ix], fluid5[(3L * g + l) * nx + ix]};
            double pM = fluid5[(4L * g + l) * nx + ix];
            double Vt[3], Tt[3];
            bool ok = nE > 0.0 && nM > 0.0 && pM > 0.0;
            for (int d = 0; d < 3 && ok; ++d) {
                Vt[d] = M[1 + d] / M[0];
                Tt[d] = M[4 + d] / M[0] - Vt[d] * Vt[d];
                ok = Tt[d] > 0.0;
            }
            if (!ok) {
#pragma omp critical
                err = ERR_DOMAIN;
                continue;
            }
            double TM = pM / (m * nM);                                   // eq. (8) closure => isotropic target (R15c)
            double scale = nM / nE;                                      // summary step 1
            double fmax = 0.0;
            for (long v = 0; v < S; ++v) { fm[v] = fe[v] * scale; fmax = std::max(fmax, fm[v]); }
            double finf = fmax;                                          // running bound (R15d)
            const long st[3] = {(long)nv[1] * nv[2], (long)nv[2], 1};
            const int maxn = std::max(nv[0], std::max(nv[1], nv[2]));
            std::vector<double> line(maxn), out(maxn), sig(maxn + 1);
            for (int d = 0; d < 3; ++d) {                                // summary step 3, x then y then z (R15b)
                double lam = std::sqrt(TM / Tt[d]);
                finf = finf / std::min(1.0, lam);
                int d1 = (d == 0) ? 1 : 0, d2 = (d == 2) ? 1 : 2;
                int n = nv[d];
                sig[0] = 0.0; sig[n] = 0.0;                              // outer faces carry no flux (R7)
                for (int k = 1; k < n; ++k) {
                    double c = vface(G, d, k);
                    double X = Vt[d] + (c - VM[d]) / lam;                 // inverse of eq. (63)
                    sig[k] = (c - X) / G.dv[d];
                }
                for (int k1 = 0; k1 < nv[d1]; ++k1)
                    for (int k2 = 0; k2 < nv[d2]; ++k2) {
                        double* base = fm + k1 * st[d1] + k2 * st[d2];
                        for (int k = 0; k < n; ++k) line[k] = base[k * st[d]];
                        remap_line(line.data(), n, sig.data(), 1, finf, limiter, out.data());
                        for (int k = 0; k < n; ++k) base[k * st[d]] = out[k];
                    }
            }
        }
    return err;
}

// --- current density, eq. (11): j = sum_s q_s M1^(s) at cell centres; if fields_yee, linearly
// interpolated to the E positions of R17.  mom: [ns][10][nyg][nx]. -----------------
void orc_current(const double* mom, int ns, const double* q, int nx, int nyg, int fields_yee,
                 int wall, double* J /*[3][nyg][nx]*/) {
    const long P = (long)nyg * nx;
    std::vector<double> jc(3 * P, 0.0);
    for (int s = 0; s < ns; ++s)
        for (int d = 0; d < 3; ++d)
            for (long c = 0; c < P; ++c) jc[d * P + c] += q[s] * mom[((long)s * 10 + 1 + d) * P + c];
    if (!fields_yee) { std::memcpy(J, jc.data(), sizeof(double) * 3 * P); return; }
    auto at = [&](int d, int j, int i) { return jc[d * P + (long)j * nx + i]; };
    for (int j = 0; j < nyg; ++j)
        for (int i = 0; i < nx; ++i) {
            int im = (i + nx - 1) % nx;
            int jm = j - 1;
            double lo = 1.0;
            if (jm < 0) { jm = nyg - 1; if (wall) lo = 0.0; }
            // on a PEC wall row (j == 0, wall) E_x and E_z are pinned to zero: J there is not used; store 0
            J[0 * P + (long)j * nx + i] = lo == 0.0 ? 0.0 : 0.5 * (at(0, jm, i) + at(0, j, i));
            J[1 * P + (long)j * nx + i] = 0.5 * (at(1, j, im) + at(1, j, i));
            J[2 * P + (long)j * nx + i] = lo == 0.0 ? 0.0 : 0.25 * (at(2, jm, im) + at(2, jm, i) + at(2, j, im) + at(2, j, i));
        }
}

// --- a10: Maxwell, 2D (d/dz = 0) Yee FDTD leapfrog, eqs. (9), (10); 8(c)-5, R17 -----------------
// nsub sub-steps of ddt = dt/nsub: E += ddt c^2 (curl B - mu0 J), then B -= ddt curl E.
// On entry E is at time T, B at T + ddt/2; J is held constant.  wall: 0 periodic in y, 1 PEC walls
// at node rows j = 0 and j = nyg (E_x = E_z = 0, B_y = 0 there).  Bavg (may be null) receives B
// linearly interpolated to the final time of E.
void orc_maxwell(double* E, double* B, const double* J, int nx, int nyg, double dx, double dy,
                 double c, double mu0, double dt, int nsub, int wall, double* Bavg) {
    const long P = (long)nyg * nx;
    const double ddt = dt / nsub;
    auto idx = [&](int d, int j, int i) { return d * P + (long)j * nx + i; };
    std::vector<double> Bold(3 * P);
    for (int sub = 0; sub < nsub; ++sub) {
        // E update, eq. (10)
        for (int j = 0; j < nyg; ++j)
            for (int i = 0; i < nx; ++i) {
                int im = (i + nx - 1) % nx;
                int jm = j - 1;
                bool onwall = false;
                if (jm < 0) { jm = nyg - 1; onwall = wall != 0; }
                double curlx = (B[idx(2, j, i)] - B[idx(2, jm, i)]) / dy;
                double curly = -(B[idx(2, j, i)] - B[idx(2, j, im)]) / dx;
                double curlz = (B[idx(1, j, i)] - B[idx(1, j, im)]) / dx - (B[idx(0, j, i)] - B[idx(0, jm, i)]) / dy;
                if (!onwall) E[idx(0, j, i)] += ddt * c * c * (curlx - mu0 * J[idx(0, j, i)]);
                else         E[idx(0, j, i)] = 0.0;
                E[idx(1, j, i)] += ddt * c * c * (curly - mu0 * J[idx(1, j, i)]);
                if (!onwall) E[idx(2, j, i)] += ddt * c * c * (curlz - mu0 * J[idx(2, j, i)]);
                else         E[idx(2, j, i)] = 0.0;
            }
        if (Bavg && sub == nsub - 1) std::memcpy(Bold.data(), B, sizeof(double) * 3 * P);
        // B update, eq. (9)
        for (int j = 0; j < nyg; ++j)
            for (int i = 0; i < nx; ++i) {
                int ip = (i + 1) % nx;
                int jp = j + 1;
                double up = 1.0;
                if (jp >= nyg) { jp = 0; if (wall) up = 0.0; }
                double dEz_dy = (up * E[idx(2, jp, i)] - E[idx(2, j, i)]) / dy;
                double dEz_dx = (E[idx(2, j, ip)] - E[idx(2, j, i)]) / dx;
                double dEy_dx = (E[idx(1, j, ip)] - E[idx(1, j, i)]) / dx;
                double dEx_dy = (up * E[idx(0, jp, i)] - E[idx(0, j, i)]) / dy;
                B[idx(0, j, i)] -= ddt * dEz_dy;
                if (wall && j == 0) B[idx(1, j, i)] = 0.0;
                else                B[idx(1, j, i)] += ddt * dEz_dx;
                B[idx(2, j, i)] -= ddt * (dEy_dx - dEx_dy);
            }
    }
    if (Bavg) for (long k = 0; k < 3 * P; ++k) Bavg[k] = 0.5 * (Bold[k] + B[k]);
}

// --- full step for one species, 8(c)-2, default order XVX (eq. 22; R2, R3) ---------------------
// stages bit mask: 1 = first spatial half (x then y), 2 = velocity step, 4 = second spatial half
// (y then x), 8 = ghost fill (sides of kind FLUID), 16 = moments into mom (may be null).
// order: 0 = XVX (eq. 22), 1 = VXV: v/2 -- x then y, full -- v/2; there stage 1 is the
// first velocity half, stage 2 the spatial step, stage 4 the second velocity half.
int orc_step(double* f, int nx, int ny, int g, const int* nv, const double* vmin, const double* vmax,
             double q, double m, double x_len, double y_len, double dt, const double* E, const double* B,
             int fields_yee, double finf, int limiter, int bc_lo, int bc_hi, const double* fluid_lo,
             const double* fluid_hi, int order, unsigned stages, double* mom) {
    const double dx = x_len / nx, dy = y_len / ny;
    const int wall = (bc_lo == BC_PERIODIC) ? 0 : 1;
    int err = ERR_OK, e;
    if (stages & 8u) {
        if (bc_lo == BC_FLUID && fluid_lo) { e = orc_ghost_fill(f, nx, ny, g, nv, vmin, vmax, m, 0, fluid_lo, limiter); if (e) err = e; }
        if (bc_hi == BC_FLUID && fluid_hi) { e = orc_ghost_fill(f, nx, ny, g, nv, vmin, vmax, m, 1, fluid_hi, limiter); if (e) err = e; }
    }
    if (order == 0) {
        if (stages & 1u) {
            orc_sweep_x(f, nx, ny, g, nv, vmin, vmax, dx, dt / 2.0, finf, limiter);
            e = orc_sweep_y(f, nx, ny, g, nv, vmin, vmax, dy, dt / 2.0, finf, limiter, bc_lo, bc_hi); if (e) err = e;
        }
        if (stages & 2u) { e = orc_vstep(f, nx, ny, g, nv, vmin, vmax, q, m, dt, E, B, fields_yee, wall, finf, limiter); if (e) err = e; }
        if (stages & 4u) {
            e = orc_sweep_y(f, nx, ny, g, nv, vmin, vmax, dy, dt / 2.0, finf, limiter, bc_lo, bc_hi); if (e) err = e;
            orc_sweep_x(f, nx, ny, g, nv, vmin, vmax, dx, dt / 2.0, finf, limiter);
        }
    } else {
        if (stages & 1u) { e = orc_vstep(f, nx, ny, g, nv, vmin, vmax, q, m, dt / 2.0, E, B, fields_yee, wall, finf, limiter); if (e) err = e; }
        if (stages & 2u) {
            orc_sweep_x(f, nx, ny, g, nv, vmin, vmax, dx, dt, finf, limiter);
            e = orc_sweep_y(f, nx, ny, g, nv, vmin, vmax, dy, dt, finf, limiter, bc_lo, bc_hi); if (e) err = e;
        }
        if (stages & 4u) { e = orc_vstep(f, nx, ny, g, nv, vmin, vmax, q, m, dt / 2.0, E, B, fields_yee, wall, finf, limiter); if (e) err = e; }
    }
    if ((stages & 16u) && mom) orc_moments(f, nx, ny, g, nv, vmin, vmax, mom);
    return err;
}

// =============================================================================================
// 3D3V ("a generalisation to the full 3-dimensional case is straightforward"):
// a third spatial direction z, periodic, nz cells of width dz.  Layout f[iz][iy_g][ix][ivx][ivy][ivz]; fields and
// moments [..][nz][ny_g][nx].  The x and y sweeps act slab by slab (the 2D functions above); the z sweep is the same
// 1D remap along z; the fields live on the 3D Yee grid (reading R24 of DESIGN.md, the standard extension of R17).
// With nz = 1 every function below reduces to its 2D counterpart bit for bit (pinned).
// =============================================================================================

// z half-sweep T(dts * v_z d/dz), periodic: sigma = v_z[ivz] * dts / dz on every face (eqs. 38, 46/47)
void orc_sweep_z(double* f, int nx, int nyg, int nz, const int* nv, const double* vmin, const double* vmax,
                 double dz, double dts, double finf, int limiter) {
    Grid G = make_grid(nx, nyg, 0, nv, vmin, vmax);
    const long S = G.nvtot;
    const long slab = (long)nyg * nx * S;           // stride between z neighbours
#pragma omp parallel
    {
        std::vector<double> line(nz), out(nz), sig(nz + 1);
#pragma omp for schedule(static)
        for (long c = 0; c < (long)nyg * nx; ++c)
            for (long v = 0; v < S; ++v) {
                int ivz = (int)(v % nv[2]);
                double s = vcen(G, 2, ivz) * dts / dz;
                for (int k = 0; k <= nz; ++k) sig[k] = s;
                double* base = f + c * S + v;
                for (int k = 0; k < nz; ++k) line[k] = base[(long)k * slab];
                remap_line(line.data(), nz, sig.data(), 0, finf, limiter, out.data());
                for (int k = 0; k < nz; ++k) base[(long)k * slab] = out[k];
            }
    }
}

// Fields at the centre of cell (ix, j, k).  3D Yee positions (R24): cell (i,j,k) spans [i dx,(i+1)dx] x [j dy,(j+1)dy] x
// [k dz,(k+1)dz]; Ex(i+1/2,j,k) Ey(i,j+1/2,k) Ez(i,j,k+1/2) Bx(i,j+1/2,k+1/2) By(i+1/2,j,k+1/2) Bz(i+1/2,j+1/2,k);
// linear interpolation to the centre; x and z periodic, row j+1 beyond the array: wrap or PEC wall value 0.
void orc_field_at_cell3d(const double* E, const double* B, int nx, int nyg, int nz, int fields_yee, int wall,
                         int ix, int j, int k, double* Ec, double* Bc) {
    const long P = (long)nz * nyg * nx;
    auto at = [&](const double* A, int d, int kk, int jj, int ii) { return A[d * P + ((long)kk * nyg + jj) * nx + ii]; };
    if (!fields_yee) {
        for (int d = 0; d < 3; ++d) { Ec[d] = at(E, d, k, j, ix); Bc[d] = at(B, d, k, j, ix); }
        return;
    }
    int ip = (ix + 1) % nx, kp = (k + 1) % nz;
    int jp = j + 1;
    double up = 1.0;
    if (jp >= nyg) { jp = 0; if (wall) up = 0.0; }
    Ec[0] = 0.25 * ((at(E, 0, k, j, ix) + up * at(E, 0, k, jp, ix)) + (at(E, 0, kp, j, ix) + up * at(E, 0, kp, jp, ix)));
    Ec[1] = 0.25 * ((at(E, 1, k, j, ix) + at(E, 1, k, j, ip)) + (at(E, 1, kp, j, ix) + at(E, 1, kp, j, ip)));
    Ec[2] = 0.25 * (at(E, 2, k, j, ix) + at(E, 2, k, j, ip) + up * at(E, 2, k, jp, ix) + up * at(E, 2, k, jp, ip));
    Bc[0] = 0.5 * (at(B, 0, k, j, ix) + at(B, 0, k, j, ip));
    Bc[1] = 0.5 * (at(B, 1, k, j, ix) + up * at(B, 1, k, jp, ix));
    Bc[2] = 0.5 * (at(B, 2, k, j, ix) + at(B, 2, kp, j, ix));
}

int orc_vstep3d(double* f, int nx, int nyg, int nz, const int* nv, const double* vmin, const double* vmax,
                double q, double m, double dt, const double* E, const double* B, int fields_yee,
                int wall, double finf, int limiter) {
    Grid G = make_grid(nx, nyg, 0, nv, vmin, vmax);
    int err = ERR_OK;
#pragma omp parallel for collapse(2) schedule(static)
    for (int k = 0; k < nz; ++k)
        for (int j = 0; j < nyg; ++j)
            for (int ix = 0; ix < nx; ++ix) {
                double Ec[3], Bc[3], t[3], s[3], h[3];
                orc_field_at_cell3d(E, B, nx, nyg, nz, fields_yee, wall, ix, j, k, Ec, Bc);
                int e = orc_boris_coeffs(Ec, Bc, q, m, dt, t, s, h);
                if (e) {
#pragma omp critical
                    err = e;
                    continue;
                }
                orc_vsweeps_block(f + (((long)k * nyg + j) * nx + ix) * G.nvtot, nv, vmin, vmax, t, s, h, finf, limiter, 0);
            }
    return err;
}

// eq. (11) on the 3D Yee grid: J at the E positions by linear interpolation of the cell-centre currents.
// mom: [ns][10][nz][nyg][nx].
void orc_current3d(const double* mom, int ns, const double* q, int nx, int nyg, int nz, int fields_yee, int wall,
                   double* J) {
    const long P = (long)nz * nyg * nx;
    std::vector<double> jc(3 * P, 0.0);
    for (int s = 0; s < ns; ++s)
        for (int d = 0; d < 3; ++d)
            for (long c = 0; c < P; ++c) jc[d * P + c] += q[s] * mom[((long)s * 10 + 1 + d) * P + c];
    if (!fields_yee) { std::memcpy(J, jc.data(), sizeof(double) * 3 * P); return; }
    auto at = [&](int d, int k, int j, int i) { return jc[d * P + ((long)k * nyg + j) * nx + i]; };
    for (int k = 0; k < nz; ++k)
        for (int j = 0; j < nyg; ++j)
            for (int i = 0; i < nx; ++i) {
                int im = (i + nx - 1) % nx, km = (k + nz - 1) % nz;
                int jm = j - 1;
                double lo = 1.0;
                if (jm < 0) { jm = nyg - 1; if (wall) lo = 0.0; }
                const long o = ((long)k * nyg + j) * nx + i;
                J[0 * P + o] = lo == 0.0 ? 0.0 : 0.25 * ((at(0, km, jm, i) + at(0, km, j, i)) + (at(0, k, jm, i) + at(0, k, j, i)));
                J[1 * P + o] = 0.25 * ((at(1, km, j, im) + at(1, km, j, i)) + (at(1, k, j, im) + at(1, k, j, i)));
                J[2 * P + o] = lo == 0.0 ? 0.0 : 0.25 * (at(2, k, jm, im) + at(2, k, jm, i) + at(2, k, j, im) + at(2, k, j, i));
            }
}

// 3D Yee FDTD leapfrog, eqs. (9), (10): nsub sub-steps of ddt = dt/nsub, E first, then B; x, z periodic; y periodic or
// PEC walls at the node rows j = 0 and j = nyg (E_x = E_z = 0, B_y = 0 there).
void orc_maxwell3d(double* E, double* B, const double* J, int nx, int nyg, int nz, double dx, double dy, double dz,
                   double c, double mu0, double dt, int nsub, int wall, double* Bavg) {
    const long P = (long)nz * nyg * nx;
    const double ddt = dt / nsub;
    auto idx = [&](int d, int k, int j, int i) { return d * P + ((long)k * nyg + j) * nx + i; };
    std::vector<double> Bold(3 * P);
    for (int sub = 0; sub < nsub; ++sub) {
        for (int k = 0; k < nz; ++k)
            for (int j = 0; j < nyg; ++j)
                for (int i = 0; i < nx; ++i) {
                    int im = (i + nx - 1) % nx, km = (k + nz - 1) % nz;
                    int jm = j - 1;
                    bool onwall = false;
                    if (jm < 0) { jm = nyg - 1; onwall = wall != 0; }
                    double curlx = (B[idx(2, k, j, i)] - B[idx(2, k, jm, i)]) / dy - (B[idx(1, k, j, i)] - B[idx(1, km, j, i)]) / dz;
                    double curly = (B[idx(0, k, j, i)] - B[idx(0, km, j, i)]) / dz - (B[idx(2, k, j, i)] - B[idx(2, k, j, im)]) / dx;
                    double curlz = (B[idx(1, k, j, i)] - B[idx(1, k, j, im)]) / dx - (B[idx(0, k, j, i)] - B[idx(0, k, jm, i)]) / dy;
                    if (!onwall) E[idx(0, k, j, i)] += ddt * c * c * (curlx - mu0 * J[idx(0, k, j, i)]);
                    else         E[idx(0, k, j, i)] = 0.0;
                    E[idx(1, k, j, i)] += ddt * c * c * (curly - mu0 * J[idx(1, k, j, i)]);
                    if (!onwall) E[idx(2, k, j, i)] += ddt * c * c * (curlz - mu0 * J[idx(2, k, j, i)]);
                    else         E[idx(2, k, j, i)] = 0.0;
                }
        if (Bavg && sub == nsub - 1) std::memcpy(Bold.data(), B, sizeof(double) * 3 * P);
        for (int k = 0; k < nz; ++k)
            for (int j = 0; j < nyg; ++j)
                for (int i = 0; i < nx; ++i) {
                    int ip = (i + 1) % nx, kp = (k + 1) % nz;
                    int jp = j + 1;
                    double up = 1.0;
                    if (jp >= nyg) { jp = 0; if (wall) up = 0.0; }
                    double dEz_dy = (up * E[idx(2, k, jp, i)] - E[idx(2, k, j, i)]) / dy;
                    double dEy_dz = (E[idx(1, kp, j, i)] - E[idx(1, k, j, i)]) / dz;
                    double dEx_dz = (E[idx(0, kp, j, i)] - E[idx(0, k, j, i)]) / dz;
                    double dEz_dx = (E[idx(2, k, j, ip)] - E[idx(2, k, j, i)]) / dx;
                    double dEy_dx = (E[idx(1, k, j, ip)] - E[idx(1, k, j, i)]) / dx;
                    double dEx_dy = (up * E[idx(0, k, jp, i)] - E[idx(0, k, j, i)]) / dy;
                    B[idx(0, k, j, i)] -= ddt * (dEz_dy - dEy_dz);
                    if (wall && j == 0) B[idx(1, k, j, i)] = 0.0;
                    else                B[idx(1, k, j, i)] -= ddt * (dEx_dz - dEz_dx);
                    B[idx(2, k, j, i)] -= ddt * (dEy_dx - dEx_dy);
                }
    }
    if (Bavg) for (long q = 0; q < 3 * P; ++q) Bavg[q] = 0.5 * (Bold[q] + B[q]);
}

// Full 3D3V step of one species.  XVX (eq. 22): x/2 y/2 z/2 -- vx vy vz -- z/2 y/2 x/2 (palindrome, R3 extended);
// VXV: v/2 -- x y z -- v/2.  y sides PERIODIC or REFLECT (no ghost rows: g = 0); stages as in orc_step.
int orc_step3d(double* f, int nx, int ny, int nz, const int* nv, const double* vmin, const double* vmax,
               double q, double m, double x_len, double y_len, double z_len, double dt, const double* E, const double* B,
               int fields_yee, double finf, int limiter, int bc_lo, int bc_hi, int order, unsigned stages, double* mom) {
    const double dx = x_len / nx, dy = y_len / ny, dz = z_len / nz;
    const int wall = (bc_lo == BC_PERIODIC) ? 0 : 1;
    Grid G = make_grid(nx, ny, 0, nv, vmin, vmax);
    const long slab = (long)ny * nx * G.nvtot;
    int err = ERR_OK, e;
    auto space = [&](double dts, bool forward) {
        if (forward) {
            for (int k = 0; k < nz; ++k) {
                orc_sweep_x(f + k * slab, nx, ny, 0, nv, vmin, vmax, dx, dts, finf, limiter);
                e = orc_sweep_y(f + k * slab, nx, ny, 0, nv, vmin, vmax, dy, dts, finf, limiter, bc_lo, bc_hi); if (e) err = e;
            }
            orc_sweep_z(f, nx, ny, nz, nv, vmin, vmax, dz, dts, finf, limiter);
        } else {
            orc_sweep_z(f, nx, ny, nz, nv, vmin, vmax, dz, dts, finf, limiter);
            for (int k = 0; k < nz; ++k) {
                e = orc_sweep_y(f + k * slab, nx, ny, 0, nv, vmin, vmax, dy, dts, finf, limiter, bc_lo, bc_hi); if (e) err = e;
                orc_sweep_x(f + k * slab, nx, ny, 0, nv, vmin, vmax, dx, dts, finf, limiter);
            }
        }
    };
    auto velocity = [&](double dtv) {
        e = orc_vstep3d(f, nx, ny, nz, nv, vmin, vmax, q, m, dtv, E, B, fields_yee, wall, finf, limiter); if (e) err = e;
    };
    if (order == 0) {
        if (stages & 1u) space(dt / 2.0, true);
        if (stages & 2u) velocity(dt);
        if (stages & 4u) space(dt / 2.0, false);
    } else {
        if (stages & 1u) velocity(dt / 2.0);
        if (stages & 2u) space(dt, true);
        if (stages & 4u) velocity(dt / 2.0);
    }
    if ((stages & 16u) && mom) orc_moments(f, nx, ny * nz, 0, nv, vmin, vmax, mom);
    return err;
}

int orc_num_threads(void) {
    int n = 1;
#ifdef _OPENMP
#pragma omp parallel
    {
#pragma omp single
        n = omp_get_num_threads();
    }
#endif
    return n;
}

}  // extern "C"
