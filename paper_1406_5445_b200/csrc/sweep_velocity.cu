// Velocity sweeps by backsubstitution (eqs. 33-35) and the table that drives them.
//
// The foot of the characteristic that ends on a face is affine in (face, transverse centre 1,
// transverse centre 2) for all three sweeps (eqs. 35, 34, 33 with the half kicks of eq. 26, R10), so
// per spatial cell the shift of face k of the line (k1, k2) is
//     sigma = c0 + c1 k + c2 k1 + c3 k2.
// A tiny kernel fills that table from E, B (a3); the ghost fill (section 4.2, eq. 63) writes the same
// table with its own affine map, so one set of sweep kernels serves both.
//
// Sweep kernels: the tile of lines is staged in shared memory, ONE THREAD PER FACE computes the flux
// of eqs. (46)/(47) (multi-cell, sign-changing shifts; zero flux through the two box faces, R7) into a
// second shared array, then every cell is updated by eq. (38).  vx: tile = all i_vx x 128 contiguous
// (i_vy,i_vz) cells.  vy+vz fused: tile = a few contiguous i_vx planes.  In place on f.
#include "vlasov_internal.cuh"

namespace vl {

// ------------------------------------------------------------------------------------------------
// a3: fields at the cell centre (R17) and the Lorentz sweep table
// ------------------------------------------------------------------------------------------------
struct TableParams {
    const double* __restrict__ E;
    const double* __restrict__ B;
    double* __restrict__ table;
    int nx, nyg, fields_yee, wall;
    double qm_half_dt;        // (q/m)(dt/2), eqs. (26), (28)
    double vmin[3], dv[3];
    double finf;
    int* err;
};

__global__ void lorentz_table_kernel(TableParams P) {
    const int cell = blockIdx.x * blockDim.x + threadIdx.x;
    const int ncell = P.nx * P.nyg;
    if (cell >= ncell) return;
    const int j = cell / P.nx, ix = cell % P.nx;
    const long PL = (long)ncell;
    double Ec[3], Bc[3];
    if (!P.fields_yee) {
        for (int d = 0; d < 3; ++d) { Ec[d] = P.E[d * PL + cell]; Bc[d] = P.B[d * PL + cell]; }
    } else {
        // cell (i,j) spans [i dx,(i+1)dx] x [j dy,(j+1)dy]; Ex(i+1/2,j) Ey(i,j+1/2) Ez(i,j)
        // Bx(i,j+1/2) By(i+1/2,j) Bz(i+1/2,j+1/2): linear interpolation to the centre
        int ip = (ix + 1) % P.nx;
        int jp = j + 1;
        double up = 1.0;
        if (jp >= P.nyg) { jp = 0; if (P.wall) up = 0.0; }
        auto at = [&](const double* A, int d, int jj, int ii) { return A[d * PL + (long)jj * P.nx + ii]; };
        Ec[0] = 0.5 * (at(P.E, 0, j, ix) + up * at(P.E, 0, jp, ix));
        Ec[1] = 0.5 * (at(P.E, 1, j, ix) + at(P.E, 1, j, ip));
        Ec[2] = 0.25 * (at(P.E, 2, j, ix) + at(P.E, 2, j, ip) + up * at(P.E, 2, jp, ix) + up * at(P.E, 2, jp, ip));
        Bc[0] = 0.5 * (at(P.B, 0, j, ix) + at(P.B, 0, j, ip));
        Bc[1] = 0.5 * (at(P.B, 1, j, ix) + up * at(P.B, 1, jp, ix));
        Bc[2] = at(P.B, 2, j, ix);
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
    P.nx = c->G.nx; P.nyg = c->G.nyg; P.fields_yee = c->G.fields_yee; P.wall = c->G.wall;
    P.qm_half_dt = (s.q / s.m) * (dt / 2.0);
    for (int d = 0; d < 3; ++d) { P.vmin[d] = s.vmin[d]; P.dv[d] = s.dv[d]; }
    P.finf = s.f_inf;
    P.err = c->errflag;
    const int ncell = P.nx * P.nyg;
    {
        Launch L(c, K_TABLE);
        lorentz_table_kernel<<<(ncell + 127) / 128, 128, 0, c->stream>>>(P);
    }
    return cudaGetLastError() == cudaSuccess ? VLASOV_OK : VLASOV_ECUDA;
}

// ------------------------------------------------------------------------------------------------
// flux through the upper face of cell k (k = 0..N-2) of a line held in shared memory
//   A[base + j*st], j = 0..N-1, zero outside (R7).  eq. (46) for sigma >= 0, eq. (47) for sigma < 0.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ double face_flux(const double* A, int base, int st, int N, int k, double sigma,
                                            double finf, int limiter) {
    const bool pos = sigma >= 0.0;
    double s = fmin(fabs(sigma), (double)(N + 3));
    int n; double b;
    split_shift(s, n, b);
    const int u = pos ? 1 : -1;
    const int j = pos ? k - n : k + 1 + n;          // foot cell
    int m = pos ? k - n + 1 : k + 1;                // whole cells between foot cell and face, ascending
    double sum = 0.0;
    for (int r = 0; r < n; ++r, ++m) sum += (m >= 0 && m < N) ? A[base + m * st] : 0.0;
    const int jm = j - u, jp = j + u;
    const double fm = (jm >= 0 && jm < N) ? A[base + jm * st] : 0.0;
    const double f0 = (j >= 0 && j < N) ? A[base + j * st] : 0.0;
    const double fp = (jp >= 0 && jp < N) ? A[base + jp * st] : 0.0;
    const double phi = sum + partial_flux(fm, f0, fp, b, finf, limiter);
    return pos ? phi : -phi;
}

// ------------------------------------------------------------------------------------------------
// a4: vx sweep.  grid = (tiles of CT contiguous (ivy,ivz) cells, spatial cells).
// ------------------------------------------------------------------------------------------------
struct VParams {
    double* __restrict__ f;
    const double* __restrict__ table;
    long S;
    int nv0, nv1, nv2;
    int cell0;        // first spatial cell (ghost-inclusive linear index) of this launch
    int limiter;
    int ct;           // columns per tile (vx kernel) / planes per tile (vyz kernel)
    int ntile;        // tiles per spatial cell
};

__global__ void __launch_bounds__(256) vsweep_x_kernel(VParams P) {
    extern __shared__ double sm[];
    const int CT = P.ct, N = P.nv0;
    const int plane = P.nv1 * P.nv2;
    double* A = sm;
    double* Phi = sm + (long)N * CT;
    const int cell = P.cell0 + blockIdx.x / P.ntile;
    const int c0 = (blockIdx.x % P.ntile) * CT;
    const int ncol = min(CT, plane - c0);
    double* fb = P.f + (long)cell * P.S + c0;
    const double* T = P.table + (long)cell * TAB;
    const double t0 = T[0], t1 = T[1], t2 = T[2], t3 = T[3], finf = T[12], scale = T[15];
    const double* fsrc = P.f + (long)T[16] * P.S + c0;
    const int tot = N * CT;
    for (int e = threadIdx.x; e < tot; e += blockDim.x) {
        int k = e / CT, c = e - k * CT;
        A[e] = c < ncol ? fsrc[(long)k * plane + c] * scale : 0.0;
    }
    __syncthreads();
    for (int e = threadIdx.x; e < tot; e += blockDim.x) {
        int k = e / CT, c = e - k * CT;
        double phi = 0.0;
        if (k < N - 1 && c < ncol) {
            int col = c0 + c;
            int k1 = col / P.nv2, k2 = col - k1 * P.nv2;
            double sigma = t0 + t1 * (k + 1) + t2 * k1 + t3 * k2;
            phi = face_flux(A, c, CT, N, k, sigma, finf, P.limiter);
        }
        Phi[e] = phi;
    }
    __syncthreads();
    for (int e = threadIdx.x; e < tot; e += blockDim.x) {
        int k = e / CT, c = e - k * CT;
        if (c < ncol) {
            double lo = k > 0 ? Phi[e - CT] : 0.0;
            fb[(long)k * plane + c] = A[e] + (lo - Phi[e]);      // eq. (38)
        }
    }
}

// ------------------------------------------------------------------------------------------------
// a5 + a6: vy sweep then vz sweep on a tile of PT contiguous i_vx planes.
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) vsweep_yz_kernel(VParams P) {
    extern __shared__ double sm[];
    const int N1 = P.nv1, N2 = P.nv2;
    const int plane = N1 * N2;
    const int cell = P.cell0 + blockIdx.x / P.ntile;
    const int p0 = (blockIdx.x % P.ntile) * P.ct;
    const int np = min(P.ct, P.nv0 - p0);
    const int tot = np * plane;
    double* A = sm;
    double* Phi = sm + (long)P.ct * plane;
    double* fb = P.f + (long)cell * P.S + (long)p0 * plane;
    const double* T = P.table + (long)cell * TAB;
    for (int e = threadIdx.x; e < tot; e += blockDim.x) A[e] = fb[e];
    __syncthreads();
    {   // vy: line along i_vy (stride N2); transverse (i_vx, i_vz)
        const double t0 = T[4], t1 = T[5], t2 = T[6], t3 = T[7], finf = T[13];
        for (int e = threadIdx.x; e < tot; e += blockDim.x) {
            int p = e / plane, r = e - p * plane;
            int k = r / N2, z = r - k * N2;
            double phi = 0.0;
            if (k < N1 - 1) {
                double sigma = t0 + t1 * (k + 1) + t2 * (p0 + p) + t3 * z;
                phi = face_flux(A, p * plane + z, N2, N1, k, sigma, finf, P.limiter);
            }
            Phi[e] = phi;
        }
        __syncthreads();
        for (int e = threadIdx.x; e < tot; e += blockDim.x) {
            int r = e % plane;
            int k = r / N2;
            double lo = k > 0 ? Phi[e - N2] : 0.0;
            A[e] = A[e] + (lo - Phi[e]);
        }
        __syncthreads();
    }
    {   // vz: contiguous lines; transverse (i_vx, i_vy)
        const double t0 = T[8], t1 = T[9], t2 = T[10], t3 = T[11], finf = T[14];
        for (int e = threadIdx.x; e < tot; e += blockDim.x) {
            int p = e / plane, r = e - p * plane;
            int y = r / N2, k = r - y * N2;
            double phi = 0.0;
            if (k < N2 - 1) {
                double sigma = t0 + t1 * (k + 1) + t2 * (p0 + p) + t3 * y;
                phi = face_flux(A, e - k, 1, N2, k, sigma, finf, P.limiter);
            }
            Phi[e] = phi;
        }
        __syncthreads();
        for (int e = threadIdx.x; e < tot; e += blockDim.x) {
            int k = e % N2;
            double lo = k > 0 ? Phi[e - 1] : 0.0;
            fb[e] = A[e] + (lo - Phi[e]);
        }
    }
}

static int g_smem_set = 0;

int launch_vsweeps(vlasov_ctx* c, const Species& s, double* f, int row0, int nrows) {
    if (nrows <= 0) return VLASOV_OK;
    if (!g_smem_set) {
        cudaFuncSetAttribute(vsweep_x_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
        cudaFuncSetAttribute(vsweep_yz_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
        g_smem_set = 1;
    }
    VParams P;
    P.f = f; P.table = c->table; P.S = s.nvtot;
    P.nv0 = s.nv[0]; P.nv1 = s.nv[1]; P.nv2 = s.nv[2];
    P.cell0 = row0 * c->G.nx;
    P.limiter = c->G.limiter;
    const int ncell = nrows * c->G.nx;
    const int plane = s.nv[1] * s.nv[2];
    {
        int ct = 128;
        while (ct > 32 && (size_t)2 * s.nv[0] * ct * 8 > 96 * 1024) ct >>= 1;
        if (ct > plane) ct = plane;
        P.ct = ct;
        size_t smem = (size_t)2 * s.nv[0] * ct * 8;
        if (smem > 200 * 1024) return VLASOV_EINVAL;
        P.ntile = (plane + ct - 1) / ct;
        Launch L(c, K_VSWEEP_X);
        vsweep_x_kernel<<<(unsigned)((long)P.ntile * ncell), 256, smem, c->stream>>>(P);
    }
    {
        int pt = (int)((32 * 1024) / ((size_t)plane * 8));
        if (pt < 1) pt = 1;
        if (pt > s.nv[0]) pt = s.nv[0];
        P.ct = pt;
        size_t smem = (size_t)2 * pt * plane * 8;
        if (smem > 200 * 1024) return VLASOV_EINVAL;
        P.ntile = (s.nv[0] + pt - 1) / pt;
        Launch L(c, K_VSWEEP_YZ);
        vsweep_yz_kernel<<<(unsigned)((long)P.ntile * ncell), 256, smem, c->stream>>>(P);
    }
    return cudaGetLastError() == cudaSuccess ? VLASOV_OK : VLASOV_ECUDA;
}

}  // namespace vl
