// a0: ghost fill at the kinetic/fluid border (section 4.2): extrapolate f from the
// Vlasov edge (zeroth order, R15a), then correct its 0th/1st/2nd moments towards the fluid state by
// a conservative remap with the affine advection field of eq. (63), one velocity
// direction after the other (R15b).  Here: moments of the edge row (moments.cu) ->
// one thread per ghost cell writes the sweep table (scale n^M/n^E, affine feet, f_infinity of R15d)
// -> the velocity sweep kernels of sweep_velocity.cu do the three remaps.
//
// a10: 2D Yee FDTD leapfrog (section 3.3, eqs. 9, 10; R17).
#include "vlasov_internal.cuh"

namespace vl {

struct GhostParams {
    const double* __restrict__ gmom;    // [11][nx] moments (+max) of the edge row
    const double* __restrict__ fluid5;  // [5][g][nx]
    double* __restrict__ table;
    int nx, ny, g, side;
    double mass;
    double vmin[3], dv[3];
    int* err;
};

__global__ void ghost_table_kernel(GhostParams P) {
    const int id = blockIdx.x * blockDim.x + threadIdx.x;
    if (id >= P.g * P.nx) return;
    const int l = id / P.nx, ix = id % P.nx;
    const int row = P.side == 0 ? P.g - 1 - l : P.g + P.ny + l;
    const int edge_row = P.side == 0 ? P.g : P.g + P.ny - 1;
    const int cell = row * P.nx + ix;
    double* T = P.table + (long)cell * TAB;
    double M[11];
    for (int k = 0; k < 11; ++k) M[k] = P.gmom[(long)k * P.nx + ix];
    const long gl = (long)P.g * P.nx;
    const double nM = P.fluid5[0 * gl + (long)l * P.nx + ix];
    const double VM[3] = {P.fluid5[1 * gl + (long)l * P.nx + ix], P.fluid5[2 * gl + (long)l * P.nx + ix],
                          P.fluid5[3 * gl + (long)l * P.nx + ix]};
    const double pM = P.fluid5[4 * gl + (long)l * P.nx + ix];
    const double nE = M[0];
    double Vt[3], Tt[3];
    bool ok = nE > 0.0 && nM > 0.0 && pM > 0.0;
    for (int d = 0; d < 3 && ok; ++d) {
        Vt[d] = M[1 + d] / M[0];                       // eq. (48) per direction (step 2 of PAPER.md:401)
        Tt[d] = M[4 + d] / M[0] - Vt[d] * Vt[d];
        ok = Tt[d] > 0.0;
    }
    if (!ok) {
        atomicCAS(P.err, 0, VLASOV_EDOMAIN);
        for (int k = 0; k < 12; ++k) T[k] = 0.0;       // leave the ghost cell as it is
        T[12] = T[13] = T[14] = 1.0; T[15] = 1.0; T[16] = (double)cell;
        return;
    }
    const double TM = pM / (P.mass * nM);              // eq. (8) closure: isotropic target (R15c)
    const double scale = nM / nE;                      // step 1 of PAPER.md:401
    double finf = M[10] * scale;                       // max of the scaled f^E; running bound (R15d)
    for (int d = 0; d < 3; ++d) {
        const double lam = sqrt(TM / Tt[d]);
        finf = finf / fmin(1.0, lam);
        const double il = 1.0 / lam;
        const double om = 1.0 - il;
        // foot X = V~ + (c - V^M)/lambda (inverse of eq. 63); sigma = (c - X)/dv, c = vmin + k dv
        T[4 * d + 0] = (P.vmin[d] * om - Vt[d] + VM[d] * il) / P.dv[d];
        T[4 * d + 1] = om;
        T[4 * d + 2] = 0.0;
        T[4 * d + 3] = 0.0;
        T[12 + d] = finf;
    }
    T[15] = scale;
    T[16] = (double)(edge_row * P.nx + ix);
}

int launch_ghost_fill(vlasov_ctx* c, const Species& s, double* f, int side) {
    const Geom& G = c->G;
    if (G.g <= 0 || !s.fluid[side]) return VLASOV_OK;
    const int edge_row = side == 0 ? G.g : G.g + G.ny - 1;
    int e = launch_moments(c, s, f, c->gmom, edge_row, 1);
    if (e) return e;
    GhostParams P;
    P.gmom = c->gmom; P.fluid5 = s.fluid[side]; P.table = c->table;
    P.nx = G.nx; P.ny = G.ny; P.g = G.g; P.side = side; P.mass = s.m;
    for (int d = 0; d < 3; ++d) { P.vmin[d] = s.vmin[d]; P.dv[d] = s.dv[d]; }
    P.err = c->errflag;
    const int n = G.g * G.nx;
    {
        Launch L(c, K_GHOST_TABLE);
        ghost_table_kernel<<<(n + 127) / 128, 128, 0, c->stream>>>(P);
    }
    if (cudaGetLastError() != cudaSuccess) return VLASOV_ECUDA;
    return launch_vsweeps(c, s, f, side == 0 ? 0 : G.g + G.ny, G.g, true);
}

// ------------------------------------------------------------------------------------------------
// Maxwell
// ------------------------------------------------------------------------------------------------
struct MaxParams {
    double* __restrict__ E;
    double* __restrict__ B;
    const double* __restrict__ J;
    double* __restrict__ Bavg;
    int nx, nyg, nz, wall;
    double dx, dy, dz, c, mu0, ddt;
    int last;
};

// E += ddt c^2 (curl B - mu0 J), eq. (10), on the Yee grid (R17; 3D: R24).  With nz = 1 every z difference
// is x - x = 0 and the update is the 2D one bit for bit.
__global__ void maxwell_E_kernel(MaxParams P) {
    const int cell = blockIdx.x * blockDim.x + threadIdx.x;
    const int ncell = P.nx * P.nyg * P.nz;
    if (cell >= ncell) return;
    const int i = cell % P.nx, j = (cell / P.nx) % P.nyg, k = cell / (P.nx * P.nyg);
    const long PL = ncell;
    const int im = (i + P.nx - 1) % P.nx, km = (k + P.nz - 1) % P.nz;
    int jm = j - 1;
    bool onwall = false;
    if (jm < 0) { jm = P.nyg - 1; onwall = P.wall != 0; }
    const double* B = P.B;
    const long c0 = cell, cjm = ((long)k * P.nyg + jm) * P.nx + i, cim = ((long)k * P.nyg + j) * P.nx + im,
               ckm = ((long)km * P.nyg + j) * P.nx + i;
    const double curlx = (B[2 * PL + c0] - B[2 * PL + cjm]) / P.dy - (B[1 * PL + c0] - B[1 * PL + ckm]) / P.dz;
    const double curly = (B[0 * PL + c0] - B[0 * PL + ckm]) / P.dz - (B[2 * PL + c0] - B[2 * PL + cim]) / P.dx;
    const double curlz = (B[1 * PL + c0] - B[1 * PL + cim]) / P.dx - (B[0 * PL + c0] - B[0 * PL + cjm]) / P.dy;
    const double kk = P.ddt * P.c * P.c;
    P.E[0 * PL + c0] = onwall ? 0.0 : P.E[0 * PL + c0] + kk * (curlx - P.mu0 * P.J[0 * PL + c0]);
    P.E[1 * PL + c0] = P.E[1 * PL + c0] + kk * (curly - P.mu0 * P.J[1 * PL + c0]);
    P.E[2 * PL + c0] = onwall ? 0.0 : P.E[2 * PL + c0] + kk * (curlz - P.mu0 * P.J[2 * PL + c0]);
}

// B -= ddt curl E, eq. (9); on the last sub-step also Bavg = (B_old + B_new)/2
__global__ void maxwell_B_kernel(MaxParams P) {
    const int cell = blockIdx.x * blockDim.x + threadIdx.x;
    const int ncell = P.nx * P.nyg * P.nz;
    if (cell >= ncell) return;
    const int i = cell % P.nx, j = (cell / P.nx) % P.nyg, k = cell / (P.nx * P.nyg);
    const long PL = ncell;
    const int ip = (i + 1) % P.nx, kp = (k + 1) % P.nz;
    int jp = j + 1;
    double up = 1.0;
    if (jp >= P.nyg) { jp = 0; if (P.wall) up = 0.0; }
    const double* E = P.E;
    const long c0 = cell, cjp = ((long)k * P.nyg + jp) * P.nx + i, cip = ((long)k * P.nyg + j) * P.nx + ip,
               ckp = ((long)kp * P.nyg + j) * P.nx + i;
    const double dEz_dy = (up * E[2 * PL + cjp] - E[2 * PL + c0]) / P.dy;
    const double dEy_dz = (E[1 * PL + ckp] - E[1 * PL + c0]) / P.dz;
    const double dEx_dz = (E[0 * PL + ckp] - E[0 * PL + c0]) / P.dz;
    const double dEz_dx = (E[2 * PL + cip] - E[2 * PL + c0]) / P.dx;
    const double dEy_dx = (E[1 * PL + cip] - E[1 * PL + c0]) / P.dx;
    const double dEx_dy = (up * E[0 * PL + cjp] - E[0 * PL + c0]) / P.dy;
    const double b0 = P.B[0 * PL + c0], b1 = P.B[1 * PL + c0], b2 = P.B[2 * PL + c0];
    const double n0 = b0 - P.ddt * (dEz_dy - dEy_dz);
    const double n1 = (P.wall && j == 0) ? 0.0 : b1 - P.ddt * (dEx_dz - dEz_dx);
    const double n2 = b2 - P.ddt * (dEy_dx - dEx_dy);
    P.B[0 * PL + c0] = n0; P.B[1 * PL + c0] = n1; P.B[2 * PL + c0] = n2;
    if (P.last && P.Bavg) {
        P.Bavg[0 * PL + c0] = 0.5 * (b0 + n0);
        P.Bavg[1 * PL + c0] = 0.5 * (b1 + n1);
        P.Bavg[2 * PL + c0] = 0.5 * (b2 + n2);
    }
}

int launch_maxwell(vlasov_ctx* c, double dt, int nsub, double* E, double* B, const double* J, double* Bavg) {
    MaxParams P;
    P.E = E; P.B = B; P.J = J; P.Bavg = Bavg;
    P.nx = c->G.nx; P.nyg = c->G.nyg; P.nz = c->G.nz; P.wall = c->G.wall;
    P.dx = c->G.dx; P.dy = c->G.dy; P.dz = c->G.dz; P.c = c->c; P.mu0 = c->mu0;
    P.ddt = dt / nsub;
    const int ncell = P.nx * P.nyg * P.nz;
    const int blocks = (ncell + 127) / 128;
    for (int sub = 0; sub < nsub; ++sub) {
        P.last = sub == nsub - 1;
        { Launch L(c, K_MAXWELL); maxwell_E_kernel<<<blocks, 128, 0, c->stream>>>(P); }
        { Launch L(c, K_MAXWELL); maxwell_B_kernel<<<blocks, 128, 0, c->stream>>>(P); }
    }
    return cudaGetLastError() == cudaSuccess ? VLASOV_OK : VLASOV_ECUDA;
}

}  // namespace vl
