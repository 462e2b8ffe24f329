// structured.cu -- SURVEY.md section 8(f), NEXT row f1: the structured cell solve ("solve_mode" = 1).
//
// The paper stores A_j dense although only 25 % of it is non-zero and names sparse cell blocks as future work
// (Eq. 41). By Eq. 8a-b, 10 and 40b
//     A_j = D - U V^T,   D = blockdiag_{(g,m)} L_{c,j,g,m}  (4 x 4 blocks, Eq. 8b),
//     V^T psi = phi      (phi[g][p] = sum_m w_m psi[g][m][p], Eq. 44),   (U phi)[g][m][p] = dx_j/4 sum_g' K_j[g][g'] phi[g'][p],
// so, exactly (Sherman-Morrison-Woodbury), the cell solve A_j x = b of Eq. 7 is
//     z = D^-1 b;   phi_z = V^T z;   y = C^-1 phi_z,  C = I - V^T D^-1 U  (4G x 4G);   x = z + D^-1 U y,
// and y = V^T x is the new scalar flux itself. Same iteration, same fixed point, same oracle (parity to
// 1e-11: cond(D), cond(C) <= ~1e3), but 4n + 16 G^2 doubles of factors per cell-solve instead of n^2.
//   st_setup   (once per dt): L^-1 of every 4 x 4 block (partial pivoting); st_wsum: W_g = sum_m w_m L^-1_{g,m}
//   st_cap     (once per dt): C = I - dx/4 (K (x) 1) W assembled on chip, inverted with partial pivoting
//   st_iterate (every iteration): a4-a7 fused, one thread per (cell, g, m)
#include "common.cuh"
#include <cooperative_groups.h>
#include <limits.h>

namespace {

// The block L_{c,j,g,m} of Eq. 8b is a 2 x 2 matrix over the numbers x + y J, J = [[0, 1], [-1, 0]] (J^2 = -I):
//     L = [[alpha, gamma/2], [-gamma, alpha + gamma]],  alpha = a I + (mu/2) J,
// and so is its inverse: every 2 x 2 sub-block of L^-1 has the form [[x, y], [-y, x]]. Rows (k,R) and (k+1/2,R) of L^-1
// therefore follow from rows (k,L) and (k+1/2,L), and only those two rows are stored and streamed: ST_LK = 8 doubles
// per block instead of 16 (the largest item of the structured path's traffic, halved). stored[0..3] = row 0,
// stored[4..7] = row 2 of the inverse inv4() computes with partial pivoting.
constexpr int ST_LK = 8;
// entry (p, c) of L^-1 from the stored rows (p, c compile-time constants in every use)
__device__ __forceinline__ double st_L(const double (&s)[ST_LK], int p, int c)
{
    const int r = (p >> 1) * 4;
    if (!(p & 1)) return s[r + c];
    return (c & 1) ? s[r + c - 1] : -s[r + c + 1];
}

// ---- once per (problem, dt): LinvT[j][k][gm], k < ST_LK (ordinate-fastest, so that the iterate kernel's loads and these
// stores are contiguous across threads). One thread per (j,g,m).
__global__ void st_setup_kernel(ProblemView P, double *__restrict__ LinvT)
{
    const int GN = P.G * P.N;
    const size_t total = (size_t)P.J * GN;
    for (size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x; e < total; e += (size_t)gridDim.x * blockDim.x) {
        const int gm = (int)(e % GN), g = gm / P.N, m = gm - g * P.N;
        const size_t j = e / GN;
        const double dx = P.dx[j], sig = P.sigma_t[j * P.G + g], v = P.v[g], mu = P.mu[m];
        double a[4][4], b[4][4];
#pragma unroll
        for (int p = 0; p < 4; ++p)
#pragma unroll
            for (int pp = 0; pp < 4; ++pp) a[p][pp] = lc_entry(p, pp, dx, sig, v, P.dt, mu);
        inv4(a, b);
#pragma unroll
        for (int k = 0; k < ST_LK; ++k) LinvT[(j * ST_LK + k) * GN + gm] = b[(k >> 2) * 2][k & 3];
    }
}

// Wg[j][g][k] = sum_m w_m (L^-1_{j,g,m})[k]. One thread per (j,g,k).
__global__ void st_wsum_kernel(ProblemView P, const double *__restrict__ LinvT, double *__restrict__ Wg)
{
    const int GN = P.G * P.N;
    const size_t total = (size_t)P.J * P.G * 16;
    for (size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x; e < total; e += (size_t)gridDim.x * blockDim.x) {
        const int k = (int)(e & 15), p = k >> 2, c = k & 3;
        const size_t jg = e >> 4;
        const int g = (int)(jg % P.G);
        const size_t j = jg / P.G;
        // entry (p, c) of L^-1 = +- a stored entry (see st_L)
        const int ks = (p >> 1) * 4 + ((p & 1) ? ((c & 1) ? c - 1 : c + 1) : c);
        const double sgn = ((p & 1) && !(c & 1)) ? -1.0 : 1.0;
        const double *src = LinvT + (j * ST_LK + ks) * GN + (size_t)g * P.N;
        double acc = 0.0;
        for (int m = 0; m < P.N; ++m) acc = fma(P.w[m], src[m], acc);
        Wg[e] = sgn * acc;
    }
}

// ---- once per (problem, dt), N a power of two <= 32: st_setup + st_wsum (+ st_cap when G = 1) in ONE launch. One thread
// per (j,g,m): the block inverse goes to LinvT; W_g = sum_m w_m L^-1 by a butterfly over the N lanes of the (cell, group),
// which leaves it in every lane; for G = 1 the capacitance matrix C = I - dx/4 K W is 4 x 4 and lane m = 0 inverts it on
// the spot (round 1: three launches, st_cap with 4 of 32 lanes active and st_wsum reading at stride G N: 0.22 ms on
// config 5 against 3 x 47 us for the iterations they serve).
template <bool G1>
__global__ void __launch_bounds__(256) st_setup_fused_kernel(ProblemView P, double *__restrict__ LinvT, double *__restrict__ Wg,
                                                             double *__restrict__ Cinv, int *info)
{
    const int GN = P.G * P.N, N = P.N;
    const size_t total = (size_t)P.J * GN;
    // whole groups of N lanes stay together: the stride is a multiple of 32 and N divides 32
    for (size_t e0 = (size_t)blockIdx.x * blockDim.x; e0 < total; e0 += (size_t)gridDim.x * blockDim.x) {
        const size_t e = e0 + threadIdx.x;
        const bool on = e < total;
        const size_t ee = on ? e : total - 1;
        const int gm = (int)(ee % GN), g = gm / N, m = gm - g * N;
        const size_t j = ee / GN;
        const double dx = P.dx[j], sig = P.sigma_t[j * P.G + g], v = P.v[g], mu = P.mu[m];
        double a[4][4], b[4][4];
#pragma unroll
        for (int p = 0; p < 4; ++p)
#pragma unroll
            for (int pp = 0; pp < 4; ++pp) a[p][pp] = lc_entry(p, pp, dx, sig, v, P.dt, mu);
        inv4(a, b);
        double st[ST_LK];
#pragma unroll
        for (int k = 0; k < ST_LK; ++k) st[k] = b[(k >> 2) * 2][k & 3];
        if (on) {
#pragma unroll
            for (int k = 0; k < ST_LK; ++k) LinvT[(j * ST_LK + k) * GN + gm] = st[k];
        }
        const double wm = on ? P.w[m] : 0.0;
        double ws[16];
#pragma unroll
        for (int k = 0; k < 16; ++k) ws[k] = wm * st_L(st, k >> 2, k & 3); // the block as the iterate kernels will see it
        for (int o = 1; o < N; o <<= 1) { // butterfly over the ordinates of the (cell, group)
#pragma unroll
            for (int k = 0; k < 16; ++k) ws[k] += __shfl_xor_sync(0xffffffffu, ws[k], o);
        }
        if (on && m == 0) {
            double *wo = Wg + (j * P.G + g) * 16;
#pragma unroll
            for (int k = 0; k < 16; ++k) wo[k] = ws[k];
            if (G1) { // C = I - dx/4 K W (4 x 4), inverted with partial pivoting; stored column-major
                const double k4 = dx * 0.25 * P.transfer[j];
                double c[4][4], ci[4][4];
#pragma unroll
                for (int p = 0; p < 4; ++p)
#pragma unroll
                    for (int pp = 0; pp < 4; ++pp) c[p][pp] = (p == pp ? 1.0 : 0.0) - k4 * ws[p * 4 + pp];
                const bool ok = inv4(c, ci);
                double *out = Cinv + j * 16;
#pragma unroll
                for (int p = 0; p < 4; ++p)
#pragma unroll
                    for (int pp = 0; pp < 4; ++pp) out[pp * 4 + p] = ok ? ci[p][pp] : 0.0;
                if (!ok) atomicMin(info, (int)j + 1);
            }
        }
    }
}

// C[(g,p)][(g',p')] = delta - (dx/4 K[g][g']) W_g[p][p']
__device__ __forceinline__ double cap_entry(const ProblemView &P, const double *__restrict__ Wg, size_t cell, int i, int c)
{
    const int g = i >> 2, p = i & 3, gc = c >> 2, pc = c & 3;
    const double k4 = P.dx[cell] * 0.25 * P.transfer[(cell * P.G + g) * P.G + gc];
    return (i == c ? 1.0 : 0.0) - k4 * Wg[(cell * P.G + g) * 16 + p * 4 + pc];
}

// ---- once per (problem, dt): C^-1 by Gauss-Jordan with partial pivoting (first maximal |entry|), one warp per cell,
// lane = row (4G <= 32), the matrix in shared memory. Stored column-major: Cinv[j][col][row].
constexpr int CAP_WARPS = 4;
constexpr int CAP_LD = 33;

__global__ void __launch_bounds__(CAP_WARPS * 32) st_cap_kernel(ProblemView P, const double *__restrict__ Wg,
                                                                double *__restrict__ Cinv, int *info)
{
    __shared__ double Wsm[CAP_WARPS][32][CAP_LD];
    __shared__ int rho_s[CAP_WARPS][32], rhoinv_s[CAP_WARPS][32];
    const int lane = threadIdx.x & 31, wp = threadIdx.x >> 5;
    const int dim = 4 * P.G;
    double(*W)[CAP_LD] = Wsm[wp];
    int *rho = rho_s[wp], *rhoinv = rhoinv_s[wp];
    const unsigned FULL = 0xffffffffu;
    for (size_t cell = (size_t)blockIdx.x * CAP_WARPS + wp; cell < (size_t)P.J; cell += (size_t)gridDim.x * CAP_WARPS) {
        for (int i = 0; i < dim; ++i)
            if (lane < dim) W[i][lane] = cap_entry(P, Wg, cell, i, lane);
        __syncwarp();
        bool used = false, singular = false;
        for (int k = 0; k < dim; ++k) {
            const double v = lane < dim ? W[lane][k] : 0.0;
            double cand = (lane < dim && !used) ? fabs(v) : -1.0;
            if (!(cand == cand)) cand = __longlong_as_double(0x7ff0000000000000LL); // NaN -> +inf: found and flagged
            int ci = lane;
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
                const double oc = __shfl_xor_sync(FULL, cand, o);
                const int oi = __shfl_xor_sync(FULL, ci, o);
                if (oc > cand || (oc == cand && oi < ci)) { cand = oc; ci = oi; }
            }
            if (!(cand > 0.0) || cand > 1.7e308) { singular = true; break; } // warp-uniform
            const int r = ci;
            const double inv = 1.0 / __shfl_sync(FULL, v, r);
            const double pr = lane < dim ? (lane == k ? 1.0 : W[r][lane]) * inv : 0.0;
            for (int i = 0; i < dim; ++i) {
                const double f = __shfl_sync(FULL, v, i);
                if (lane < dim) W[i][lane] = (i == r) ? pr : fma(-f, pr, lane == k ? 0.0 : W[i][lane]);
            }
            if (lane == r) used = true;
            if (lane == 0) { rho[k] = r; rhoinv[r] = k; }
            __syncwarp();
        }
        double *out = Cinv + cell * dim * dim;
        if (singular) {
            if (lane == 0) atomicMin(info, (int)cell + 1);
            for (int e = lane; e < dim * dim; e += 32) out[e] = 0.0;
        } else { // Cinv[kappa][rho_j] = W[rho_kappa][j]: un-scrambles the implicit row exchange
            for (int jc = 0; jc < dim; ++jc)
                if (lane < dim) out[(size_t)rho[jc] * dim + rhoinv[lane]] = W[lane][jc];
        }
        __syncwarp();
    }
}

// ---- every iteration: a4 (gather + RHS), a5 (structured solve), a6 (phi), a7 (residual), one thread per (cell, g, m).
// A CTA works on CPB = 256 / (G N) consecutive cells at a time. Loads are contiguous across the threads of a cell
// (c_j and Psi: 32 bytes per thread; LinvT: ordinate-fastest; Cinv: column-major, one row per thread).
constexpr int ST_THREADS = 256;

struct StParams {
    const double *LinvT, *Cinv, *dx, *transfer;
};

// GC = G when G is 1, 2, 4 or 8 (the 4G rows of a cell then sit inside one warp, so the three small steps between
// z and x need only __syncwarp, and for G <= 4 the thread's row of C^-1, its row of K and dx are loaded up front,
// together with everything else, so that a CTA waits for HBM once); GC = 0: any G, CTA-wide barriers.
// COHERENT: Psi^(l) and phi^(l) were written by other CTAs of the SAME launch (st_iterate_multi_kernel): read past L1.
template <bool COHERENT> __device__ __forceinline__ double ld_iter(const double *p) { return COHERENT ? __ldcg(p) : *p; }

template <bool WANT_L2, int GC, bool COHERENT>
__device__ __forceinline__ void st_iterate_body(const IterParams &P, const StParams &S, double *st_smem)
{
    const int N = P.N, G = GC > 0 ? GC : P.G, J = P.J, n = P.n, GN = G * N, G4 = 4 * G;
    constexpr bool PRE = GC > 0 && GC <= 4;
    constexpr int GP = PRE ? GC : 1;
    const int CPB = ST_THREADS / GN;
    double *mu_s = st_smem;                   // [N]
    double *w_s = mu_s + N;                   // [N]
    double *wz = w_s + N;                     // [CPB][GN][4]   w_m z
    double *phiz = wz + (size_t)CPB * GN * 4; // [CPB][4G]
    double *ys = phiz + (size_t)CPB * G4;     // [CPB][4G]
    double *ss = ys + (size_t)CPB * G4;       // [CPB][4G]
    const int tid = threadIdx.x, lane = tid & 31;
    for (int i = tid; i < N; i += ST_THREADS) { mu_s[i] = P.mu[i]; w_s[i] = P.w[i]; }

    const int a = tid / GN, gm = tid - a * GN, g = gm / N, m = gm - g * N;
    const bool lane_on = tid < CPB * GN;
    const int rows = CPB * G4;
    double rmax = 0.0, l2 = 0.0;
    auto small_sync = [&]() {
        if (GC > 0) __syncwarp();
        else __syncthreads();
    };

    // ordering: all cells (ncolors = 1, Jacobi) or the cells of one colour (ncolors = 2: j = 2 i + color), in place
    const int NC = P.ncolors, Jc = (J - P.color + NC - 1) / NC;
    for (int base = blockIdx.x * CPB; base < Jc; base += gridDim.x * CPB) {
        const int j = NC * (base + a) + P.color;
        const bool on = lane_on && base + a < Jc;
        double L[ST_LK], z[4], b[4], v0 = 0.0, v1 = 0.0, mu = 1.0;
        // ---- all global loads of this batch up front
        if (on) {
            const double2 c01 = *reinterpret_cast<const double2 *>(P.c + (size_t)j * n + gm * 4);
            const double2 c23 = *reinterpret_cast<const double2 *>(P.c + (size_t)j * n + gm * 4 + 2);
            b[0] = c01.x; b[1] = c01.y; b[2] = c23.x; b[3] = c23.y;
            mu = P.mu[m];
            const double *self = P.psi_old + (size_t)j * n;
            // a4: incident edge fluxes from Psi^(l) (Eq. 9c-d; closures Eq. 5a-b)
            if (mu > 0.0) { // rows (k,L), (k+1/2,L): upstream = (j-1, R)
                if (j > 0) { v0 = ld_iter<COHERENT>(self - n + gm * 4 + 1); v1 = ld_iter<COHERENT>(self - n + gm * 4 + 3); }
                else if (P.bc_left == OCI_BC_REFLECTIVE) {
                    v0 = ld_iter<COHERENT>(self + (g * N + (N - 1 - m)) * 4 + 0); v1 = ld_iter<COHERENT>(self + (g * N + (N - 1 - m)) * 4 + 2);
                } else if (P.bc_left == OCI_BC_PRESCRIBED) { v0 = P.inc_left[gm * 2]; v1 = P.inc_left[gm * 2 + 1]; }
            } else {        // rows (k,R), (k+1/2,R): upstream = (j+1, L)
                if (j < J - 1) { v0 = ld_iter<COHERENT>(self + n + gm * 4 + 0); v1 = ld_iter<COHERENT>(self + n + gm * 4 + 2); }
                else if (P.bc_right == OCI_BC_REFLECTIVE) {
                    v0 = ld_iter<COHERENT>(self + (g * N + (N - 1 - m)) * 4 + 1); v1 = ld_iter<COHERENT>(self + (g * N + (N - 1 - m)) * 4 + 3);
                } else if (P.bc_right == OCI_BC_PRESCRIBED) { v0 = P.inc_right[gm * 2]; v1 = P.inc_right[gm * 2 + 1]; }
            }
            const double *Lp = S.LinvT + (size_t)j * ST_LK * GN + gm;
#pragma unroll
            for (int k = 0; k < ST_LK; ++k) L[k] = Lp[(size_t)k * GN];
        }
        double Cr[4 * GP], Kr[GP], dxq = 0.0, phi_old = 0.0; // this thread's (first) row of the 4G-system
        if (PRE && tid < rows && base + tid / G4 < Jc) {
            const int a2 = tid / G4, r2 = tid - a2 * G4, j2 = NC * (base + a2) + P.color;
            const double *Cp = S.Cinv + (size_t)j2 * G4 * G4 + r2;
#pragma unroll
            for (int cc = 0; cc < 4 * GP; ++cc) Cr[cc] = Cp[(size_t)cc * G4];
            const double *Kp = S.transfer + ((size_t)j2 * G + (r2 >> 2)) * G;
#pragma unroll
            for (int gc = 0; gc < GP; ++gc) Kr[gc] = Kp[gc];
            dxq = S.dx[j2] * 0.25;
            phi_old = ld_iter<COHERENT>(P.phi + (size_t)j2 * G4 + r2);
        }
        __syncthreads(); // previous batch done with the shared arrays (and mu_s / w_s loaded)
        if (on) {
            if (mu > 0.0) { b[0] = fma(mu, v0, b[0]); b[2] = fma(mu, v1, b[2]); }
            else { b[1] = fma(-mu, v0, b[1]); b[3] = fma(-mu, v1, b[3]); }
            const double wm = w_s[m];
#pragma unroll
            for (int p = 0; p < 4; ++p) { // z = D^-1 b
                z[p] = fma(st_L(L, p, 3), b[3], fma(st_L(L, p, 2), b[2], fma(st_L(L, p, 1), b[1], st_L(L, p, 0) * b[0])));
                wz[(size_t)tid * 4 + p] = wm * z[p];
            }
        }
        __syncthreads();
        // ---- phi_z = V^T z, y = C^-1 phi_z = phi^(l+1) (a6), residual (a7), s = dx/4 K y: one (cell, g, p) row per
        // thread-iteration (4G rows per cell; 4G > G N when N = 2, hence the loops)
        for (int t2 = tid; t2 < rows; t2 += ST_THREADS) {
            const int a2 = t2 / G4, r2 = t2 - a2 * G4;
            if (base + a2 < Jc) {
                const int g2 = r2 >> 2, p2 = r2 & 3;
                const double *src = wz + ((size_t)a2 * GN + g2 * N) * 4 + p2;
                double acc = 0.0;
                for (int mm = 0; mm < N; ++mm) acc += src[mm * 4];
                phiz[t2] = acc;
            }
        }
        small_sync();
        for (int t2 = tid; t2 < rows; t2 += ST_THREADS) {
            const int a2 = t2 / G4, r2 = t2 - a2 * G4, j2 = NC * (base + a2) + P.color;
            if (base + a2 < Jc) {
                const double *pz = phiz + a2 * G4;
                double y = 0.0, po;
                if (PRE && t2 == tid) {
#pragma unroll
                    for (int cc = 0; cc < 4 * GP; ++cc) y = fma(Cr[cc], pz[cc], y);
                    po = phi_old;
                } else {
                    const double *Cp = S.Cinv + (size_t)j2 * G4 * G4 + r2;
                    for (int cc = 0; cc < G4; ++cc) y = fma(Cp[(size_t)cc * G4], pz[cc], y);
                    po = ld_iter<COHERENT>(P.phi + (size_t)j2 * G4 + r2);
                }
                ys[t2] = y;
                P.phi[(size_t)j2 * G4 + r2] = y;
                const double d = fabs(y - po);
                rmax = (d > rmax || !(d == d)) ? d : rmax;
            }
        }
        small_sync();
        for (int t2 = tid; t2 < rows; t2 += ST_THREADS) {
            const int a2 = t2 / G4, r2 = t2 - a2 * G4, j2 = NC * (base + a2) + P.color;
            if (base + a2 < Jc) {
                const int g2 = r2 >> 2, p2 = r2 & 3;
                const double *yy = ys + a2 * G4 + p2;
                double acc = 0.0;
                if (PRE && t2 == tid) {
#pragma unroll
                    for (int gc = 0; gc < GP; ++gc) acc = fma(Kr[gc], yy[gc * 4], acc);
                    ss[t2] = dxq * acc;
                } else {
                    const double *Kp = S.transfer + ((size_t)j2 * G + g2) * G;
                    for (int gc = 0; gc < G; ++gc) acc = fma(Kp[gc], yy[gc * 4], acc);
                    ss[t2] = S.dx[j2] * 0.25 * acc;
                }
            }
        }
        __syncthreads();
        // ---- x = z + D^-1 U y
        if (on) {
            const double *sv = ss + a * G4 + g * 4;
            const double s0 = sv[0], s1 = sv[1], s2 = sv[2], s3 = sv[3];
            double x[4];
#pragma unroll
            for (int p = 0; p < 4; ++p)
                x[p] = fma(st_L(L, p, 3), s3, fma(st_L(L, p, 2), s2, fma(st_L(L, p, 1), s1, fma(st_L(L, p, 0), s0, z[p]))));
            double *out = P.psi_new + (size_t)j * n + gm * 4;
            if (WANT_L2) {
                const double *old = P.psi_old + (size_t)j * n + gm * 4;
#pragma unroll
                for (int p = 0; p < 4; ++p) { const double d = x[p] - ld_iter<COHERENT>(old + p); l2 = fma(d, d, l2); }
            }
            *reinterpret_cast<double2 *>(out) = make_double2(x[0], x[1]);
            *reinterpret_cast<double2 *>(out + 2) = make_double2(x[2], x[3]);
        }
    }
    rmax = warp_max(rmax);
    if (lane == 0) atomicMax(P.resid_inf, resid_bits(rmax));
    if (WANT_L2) {
        l2 = warp_sum(l2);
        if (lane == 0) atomicAdd(P.resid_l2, l2);
    }
}


template <bool WANT_L2, int GC>
__global__ void __launch_bounds__(ST_THREADS, 3) st_iterate_kernel(const IterParams P, const StParams S)
{
    if (stop_reached(P.stop)) return;
    if (blockIdx.x == 0 && threadIdx.x == 0) *P.stop.executed = P.stop.slot + 1;
    extern __shared__ __align__(16) double st_smem[];
    st_iterate_body<WANT_L2, GC, false>(P, S, st_smem);
}

// persistent multi-iteration kernel for problems whose factors stay in L2. One COOPERATIVE launch
// runs up to n_iters block-Jacobi iterations, a grid-wide barrier between them (every CTA keeps its cells, the two
// Psi buffers alternate, data written by other CTAs is read past the L1), with the same device-side stop: after the
// barrier every thread of the grid reads the same residual slot and takes the same decision. Replaces n_iters launches
// of ~4 us of fixed cost each by n_iters grid barriers.
struct StMulti {
    int n_iters, slot0, check_between, rule;
    double tol;
    unsigned long long *resid_inf; // history base (slot 0)
    double *resid_l2;
    int *executed;
};

template <bool WANT_L2, int GC>
__global__ void __launch_bounds__(ST_THREADS, 3) st_iterate_multi_kernel(const IterParams P, const StParams S, const StMulti M)
{
    extern __shared__ __align__(16) double st_smem[];
    cooperative_groups::grid_group grid = cooperative_groups::this_grid();
    IterParams Q = P;
    for (int it = 0; it < M.n_iters; ++it) {
        const int slot = M.slot0 + it;
        if (M.check_between && it > 0) {
            StopCheck st;
            st.prev_inf = M.resid_inf + slot - 1;
            st.prev_l2 = M.resid_l2 + slot - 1;
            st.prev2_l2 = slot >= 2 ? M.resid_l2 + slot - 2 : nullptr;
            st.tol = M.tol; st.rule = M.rule; st.slot = slot; st.executed = M.executed;
            if (stop_reached_t<true>(st)) break; // same values everywhere: the whole grid leaves together
        }
        if (blockIdx.x == 0 && threadIdx.x == 0) *M.executed = slot + 1;
        Q.psi_old = (it & 1) ? P.psi_new : P.psi_old;
        Q.psi_new = (it & 1) ? const_cast<double *>(P.psi_old) : P.psi_new;
        Q.resid_inf = M.resid_inf + slot;
        Q.resid_l2 = M.resid_l2 + slot;
        st_iterate_body<WANT_L2, GC, true>(Q, S, st_smem);
        grid.sync();
    }
}

// ============================================================================================================
// Persistent, bulk-copy-pipelined version of st_iterate_kernel (the production kernel of solve_mode 1).
// ============================================================================================================
// Same arithmetic, thread for thread. One CTA per SM owns a contiguous range of cells and walks it in batches of
// CPB = 256 / (G N) cells; per batch one producer thread issues four 1-D bulk async copies (the batch's 4x4 block
// inverses, c_j, Psi^(l) of the batch and its two neighbour cells, C^-1 -- each contiguous in HBM by construction of
// the layouts) into a ring of `stages` shared-memory stages guarded by mbarriers, so that HBM stays busy while the
// 256 consumer threads work out of shared memory. The blocks are re-read from shared memory for x = z + D^-1 U y
// instead of being held in registers across the barriers.
constexpr int STP_MAX_STAGES = 6;

struct StStage {                // element offsets inside one stage (all multiples of 2 doubles)
    int Lt, cs, nb, Ci, doubles;
};

__host__ __device__ inline StStage st_stage_layout(int N, int G, int CT)
{
    const int GN = G * N, n = 4 * GN, G4 = 4 * G, CPB = CT / GN;
    StStage s;
    s.Lt = 0;
    s.cs = s.Lt + CPB * ST_LK * GN;
    s.nb = s.cs + CPB * n;
    s.Ci = s.nb + (CPB + 2) * n;
    s.doubles = (s.Ci + CPB * G4 * G4 + 15) & ~15; // stages stay 128-byte aligned
    return s;
}

// CT = consumer threads per CTA (256, or 128 so that four CTAs share an SM); one more warp holds the producer thread.
template <bool WANT_L2, int GC, int CT>
__global__ void __launch_bounds__(CT + 32, CT == 256 ? 2 : 4) st_iterate_pipe_kernel(const IterParams P, const StParams S, int stages,
                                                                                     int warp_local)
{
    pdl_launch_dependents(); // (see launch_pdl: everything up to pdl_wait() below touches constant inputs only)
    extern __shared__ __align__(128) unsigned char stp_smem[];
    const int N = P.N, G = GC > 0 ? GC : P.G, J = P.J, n = P.n, GN = G * N, G4 = 4 * G;
    constexpr int STP_CONSUMERS = CT, STP_THREADS = CT + 32;
    const int CPB = CT / GN;
    const StStage lay = st_stage_layout(N, G, CT);
    uint64_t *full = reinterpret_cast<uint64_t *>(stp_smem);
    uint64_t *empty = full + STP_MAX_STAGES;
    double *mu_s = reinterpret_cast<double *>(empty + STP_MAX_STAGES); // [N]
    double *w_s = mu_s + N;                                           // [N]
    double *wz = w_s + N;                                             // [CPB][GN][4]
    double *phiz = wz + (size_t)CPB * GN * 4;                         // [CPB][4G]
    double *ys = phiz + (size_t)CPB * G4;                             // [CPB][4G]
    double *ss = ys + (size_t)CPB * G4;                               // [CPB][4G]
    // prescribed incident fluxes in shared memory: a global load inside the batch body would share a scoreboard slot
    // with the role-2 prefetch loads below and make every batch wait for them (ncu: 19 % of the samples, long_sb)
    double *incl_s = ss + (size_t)CPB * G4;                           // [G N][2]
    double *incr_s = incl_s + 2 * GN;                                 // [G N][2]
    size_t off = (size_t)((unsigned char *)(incr_s + 2 * GN) - stp_smem);
    off = (off + 127) & ~(size_t)127;
    double *ring = reinterpret_cast<double *>(stp_smem + off);        // stages x lay.doubles

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid == 0) {
        for (int s = 0; s < stages; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], STP_CONSUMERS / 32); }
        fence_mbar_init();
    }
    for (int i = tid; i < N; i += STP_THREADS) { mu_s[i] = P.mu[i]; w_s[i] = P.w[i]; }
    for (int i = tid; i < 2 * GN; i += STP_THREADS) {
        incl_s[i] = P.bc_left == OCI_BC_PRESCRIBED ? P.inc_left[i] : 0.0;
        incr_s[i] = P.bc_right == OCI_BC_PRESCRIBED ? P.inc_right[i] : 0.0;
    }
    __syncthreads();
    pdl_wait(); // the previous iteration (or whatever precedes on the stream) is complete from here on
    if (stop_reached(P.stop)) return;
    if (blockIdx.x == 0 && threadIdx.x == 0) *P.stop.executed = P.stop.slot + 1;

    const int cell0 = (int)(((long long)J * blockIdx.x) / gridDim.x);
    const int cell1 = (int)(((long long)J * (blockIdx.x + 1)) / gridDim.x);
    // successive iterations walk the range in opposite directions (P.reverse, see oci_iterate_wpc_kernel): what a CTA
    // touched last is what it asks for first next time, while it is still in the L2 -- here an iteration's whole stream
    // (164 MB on config 5) is of the order of the L2
    const int nbatch = (cell1 - cell0 + CPB - 1) / CPB;
    auto batch_first = [&](int bi) { return cell0 + CPB * (P.reverse ? nbatch - 1 - bi : bi); };

    if (warp == STP_CONSUMERS / 32) {
        // ===================== producer =====================================================================
        if (lane == 0) {
            int st = 0;
            uint32_t ph = 0;
            for (int bi = 0; bi < nbatch; ++bi) {
                const int gb = batch_first(bi);
                const int nb = min(CPB, cell1 - gb);
                mbar_wait(&empty[st], ph ^ 1);
                double *base = ring + (size_t)st * lay.doubles;
                const int lo = max(gb - 1, 0), hi = min(gb + nb, J - 1);
                const uint32_t bL = (uint32_t)((size_t)nb * ST_LK * GN * sizeof(double));
                const uint32_t bc = (uint32_t)((size_t)nb * n * sizeof(double));
                const uint32_t bn = (uint32_t)((size_t)(hi - lo + 1) * n * sizeof(double));
                const uint32_t bC = (uint32_t)((size_t)nb * G4 * G4 * sizeof(double));
                mbar_arrive_expect_tx(&full[st], bL + bc + bn + bC);
                bulk_g2s(base + lay.Lt, S.LinvT + (size_t)gb * ST_LK * GN, bL, &full[st]);
                bulk_g2s(base + lay.cs, P.c + (size_t)gb * n, bc, &full[st]);
                bulk_g2s(base + lay.nb + (size_t)(lo - (gb - 1)) * n, P.psi_old + (size_t)lo * n, bn, &full[st]);
                bulk_g2s(base + lay.Ci, S.Cinv + (size_t)gb * G4 * G4, bC, &full[st]);
                if (++st == stages) { st = 0; ph ^= 1; }
            }
        }
        return;
    }

    // ========================= consumers ====================================================================
    const int a = tid / GN, gm = tid - a * GN, g = gm / N, m = gm - g * N;
    const bool lane_on = tid < CPB * GN;
    const int rows = CPB * G4;
    double rmax = 0.0, l2 = 0.0;
    auto consumer_sync = [&]() { asm volatile("bar.sync 1, %0;" ::"n"(STP_CONSUMERS) : "memory"); };
    auto small_sync = [&]() {
        if (GC > 0) __syncwarp();
        else consumer_sync();
    };
    // butterfly reduction over the ordinates: N a power of two <= 32 (groups of N lanes never straddle a warp then)
    const bool shfl_reduce = N <= 32 && (N & (N - 1)) == 0;
    // warp_local (host: GC > 0, N a power of two >= 4, G N <= 32): a cell's G N threads sit inside one warp and ALSO do
    // the cell's 4G-row steps (thread (a, gm) takes row gm < 4G), so every exchange of a batch is warp-local and the
    // batch needs no CTA barrier at all (ncu on the previous version: 28 % of the warp samples in bar.sync). For G = 1
    // there is not even an exchange: the butterfly leaves phi_z in every lane, and each lane applies the 4 x 4 C^-1.
    const bool wl = GC > 0 && warp_local != 0;
    double Kr_n[GC > 0 ? GC : 1], dxq_n = 0.0, phi_old_n = 0.0;
    auto load_role2 = [&](int gb_, int nb_) {
        if (wl) {
            if (a < nb_ && lane_on && (gm < G4 || GC == 1)) {
                const int j2 = gb_ + a, r2 = gm < G4 ? gm : 0;
                const double *Kp = S.transfer + ((size_t)j2 * G + (r2 >> 2)) * G;
#pragma unroll
                for (int gc = 0; gc < (GC > 0 ? GC : 1); ++gc) Kr_n[gc] = Kp[gc];
                dxq_n = S.dx[j2];
                if (gm < G4) phi_old_n = P.phi[(size_t)j2 * G4 + gm];
            }
        } else if (GC > 0 && tid < rows && tid / G4 < nb_) {
            const int a2 = tid / G4, r2 = tid - a2 * G4, j2 = gb_ + a2;
            const double *Kp = S.transfer + ((size_t)j2 * G + (r2 >> 2)) * G;
#pragma unroll
            for (int gc = 0; gc < (GC > 0 ? GC : 1); ++gc) Kr_n[gc] = Kp[gc];
            dxq_n = S.dx[j2]; // used (x 0.25) one batch later: nothing here waits for the load
            phi_old_n = P.phi[(size_t)j2 * G4 + r2];
        }
    };
    if (nbatch > 0) load_role2(batch_first(0), min(CPB, cell1 - batch_first(0)));
    int st = 0;
    uint32_t ph = 0;
    for (int bi = 0; bi < nbatch; ++bi) {
        const int gb = batch_first(bi);
        const int nb = min(CPB, cell1 - gb);
        const double *base = ring + (size_t)st * lay.doubles;
        const int j = gb + a;
        const bool on = lane_on && a < nb;
        // role-2 data that is not worth a bulk copy (this thread's row of K, dx, phi^(l)): plain loads, issued one
        // batch ahead so that their latency never sits between two barriers
        double Kr[GC > 0 ? GC : 1], dxq = dxq_n, phi_old = phi_old_n;
#pragma unroll
        for (int gc = 0; gc < (GC > 0 ? GC : 1); ++gc) Kr[gc] = Kr_n[gc];
        if (bi + 1 < nbatch) load_role2(batch_first(bi + 1), min(CPB, cell1 - batch_first(bi + 1)));
        mbar_wait(&full[st], ph);
        double z[4];
        // the two stored rows of this thread's block inverse: in registers, except for G = 8, whose instantiation has
        // none to spare (it re-reads them from the stage)
        constexpr bool L_IN_REGS = GC != 8;
        const double *Lp = base + lay.Lt + (size_t)a * ST_LK * GN + gm;
        double Ls[ST_LK];
        if (L_IN_REGS) {
#pragma unroll
            for (int k = 0; k < ST_LK; ++k) Ls[k] = on ? Lp[k * GN] : 0.0;
        }
        auto Lent = [&](int p, int c) -> double {
            if (L_IN_REGS) return st_L(Ls, p, c);
            const int r = (p >> 1) * 4;
            if (!(p & 1)) return Lp[(r + c) * GN];
            return (c & 1) ? Lp[(r + c - 1) * GN] : -Lp[(r + c + 1) * GN];
        };
        if (on) {
            const double2 *cp = reinterpret_cast<const double2 *>(base + lay.cs + (size_t)a * n + gm * 4);
            const double2 c01 = cp[0], c23 = cp[1];
            double b[4] = {c01.x, c01.y, c23.x, c23.y};
            const double mu = mu_s[m];
            const double *self = base + lay.nb + (size_t)(a + 1) * n;
            double v0 = 0.0, v1 = 0.0;
            // a4: incident edge fluxes from Psi^(l) (Eq. 9c-d; closures Eq. 5a-b)
            if (mu > 0.0) {
                if (j > 0) { // 16-byte loads: two-way instead of eight-way bank conflicts at the 32-byte thread stride
                    const double2 *up = reinterpret_cast<const double2 *>(self - n + gm * 4);
                    v0 = up[0].y; v1 = up[1].y;
                }
                else if (P.bc_left == OCI_BC_REFLECTIVE) {
                    v0 = self[(g * N + (N - 1 - m)) * 4 + 0]; v1 = self[(g * N + (N - 1 - m)) * 4 + 2];
                } else if (P.bc_left == OCI_BC_PRESCRIBED) { v0 = incl_s[gm * 2]; v1 = incl_s[gm * 2 + 1]; }
                b[0] = fma(mu, v0, b[0]);
                b[2] = fma(mu, v1, b[2]);
            } else {
                if (j < J - 1) {
                    const double2 *up = reinterpret_cast<const double2 *>(self + n + gm * 4);
                    v0 = up[0].x; v1 = up[1].x;
                }
                else if (P.bc_right == OCI_BC_REFLECTIVE) {
                    v0 = self[(g * N + (N - 1 - m)) * 4 + 1]; v1 = self[(g * N + (N - 1 - m)) * 4 + 3];
                } else if (P.bc_right == OCI_BC_PRESCRIBED) { v0 = incr_s[gm * 2]; v1 = incr_s[gm * 2 + 1]; }
                b[1] = fma(-mu, v0, b[1]);
                b[3] = fma(-mu, v1, b[3]);
            }
#pragma unroll
            for (int p = 0; p < 4; ++p) // z = D^-1 b
                z[p] = fma(Lent(p, 3), b[3], fma(Lent(p, 2), b[2], fma(Lent(p, 1), b[1], Lent(p, 0) * b[0])));
        }
        // phi_z = V^T z: the N ordinates of a (cell, group) are N consecutive lanes -> butterfly when N is a power of two
        double q[4];
        {
            const double wm = on ? w_s[m] : 0.0;
#pragma unroll
            for (int p = 0; p < 4; ++p) q[p] = on ? wm * z[p] : 0.0;
            if (shfl_reduce) {
                for (int o = N >> 1; o > 0; o >>= 1) {
#pragma unroll
                    for (int p = 0; p < 4; ++p) q[p] += __shfl_xor_sync(0xffffffffu, q[p], o);
                }
                if (on && m == 0) {
                    double2 *dst = reinterpret_cast<double2 *>(phiz + a * G4 + g * 4);
                    dst[0] = make_double2(q[0], q[1]);
                    dst[1] = make_double2(q[2], q[3]);
                }
            } else if (on) {
                double2 *dst = reinterpret_cast<double2 *>(wz + (size_t)tid * 4);
                dst[0] = make_double2(q[0], q[1]);
                dst[1] = make_double2(q[2], q[3]);
            }
        }
        if (wl) {
            // ================= warp-local steps: y = C^-1 phi_z = phi^(l+1), residual, s = dx/4 K y, x = z + D^-1 U y =========
            double s4[4] = {0.0, 0.0, 0.0, 0.0};
            if (GC == 1) {
                if (on) {
                    const double2 *C2 = reinterpret_cast<const double2 *>(base + lay.Ci + (size_t)a * 16);
                    double y[4] = {0.0, 0.0, 0.0, 0.0};
#pragma unroll
                    for (int cc = 0; cc < 4; ++cc) { // column cc of the column-major 4 x 4 C^-1
                        const double2 c01 = C2[2 * cc], c23 = C2[2 * cc + 1];
                        y[0] = fma(c01.x, q[cc], y[0]); y[1] = fma(c01.y, q[cc], y[1]);
                        y[2] = fma(c23.x, q[cc], y[2]); y[3] = fma(c23.y, q[cc], y[3]);
                    }
                    if (gm < 4) {
                        const double yv = gm == 0 ? y[0] : (gm == 1 ? y[1] : (gm == 2 ? y[2] : y[3]));
                        P.phi[(size_t)j * 4 + gm] = yv;
                        const double d = fabs(yv - phi_old);
                        rmax = (d > rmax || !(d == d)) ? d : rmax;
                    }
#pragma unroll
                    for (int p = 0; p < 4; ++p) { double acc = 0.0; acc = fma(Kr[0], y[p], acc); s4[p] = dxq * 0.25 * acc; }
                }
            } else { // (phi_z of the cell's groups was written by the m == 0 lanes above)
                __syncwarp();
                if (on && gm < G4) {
                    const double *Cp = base + lay.Ci + (size_t)a * G4 * G4 + gm;
                    const double *pz = phiz + a * G4;
                    double y = 0.0;
                    for (int cc = 0; cc < G4; ++cc) y = fma(Cp[cc * G4], pz[cc], y);
                    ys[a * G4 + gm] = y;
                    P.phi[(size_t)j * G4 + gm] = y;
                    const double d = fabs(y - phi_old);
                    rmax = (d > rmax || !(d == d)) ? d : rmax;
                }
                __syncwarp();
                if (on && gm < G4) {
                    const double *yy = ys + a * G4 + (gm & 3);
                    double acc = 0.0;
#pragma unroll
                    for (int gc = 0; gc < (GC > 0 ? GC : 1); ++gc) acc = fma(Kr[gc], yy[gc * 4], acc);
                    ss[a * G4 + gm] = dxq * 0.25 * acc;
                }
                __syncwarp();
                if (on) {
                    const double *sv = ss + a * G4 + g * 4;
                    s4[0] = sv[0]; s4[1] = sv[1]; s4[2] = sv[2]; s4[3] = sv[3];
                }
            }
            if (on) {
                double x[4];
#pragma unroll
                for (int p = 0; p < 4; ++p)
                    x[p] = fma(Lent(p, 3), s4[3], fma(Lent(p, 2), s4[2], fma(Lent(p, 1), s4[1], fma(Lent(p, 0), s4[0], z[p]))));
                if (WANT_L2) {
                    const double *old = base + lay.nb + (size_t)(a + 1) * n + gm * 4;
#pragma unroll
                    for (int p = 0; p < 4; ++p) { const double d = x[p] - old[p]; l2 = fma(d, d, l2); }
                }
                double *out = P.psi_new + (size_t)j * n + gm * 4;
                *reinterpret_cast<double2 *>(out) = make_double2(x[0], x[1]);
                *reinterpret_cast<double2 *>(out + 2) = make_double2(x[2], x[3]);
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(&empty[st]); // this warp is done with the stage
            if (++st == stages) { st = 0; ph ^= 1; }
            continue;
        }
        consumer_sync();
        for (int t2 = tid; !shfl_reduce && t2 < rows; t2 += STP_CONSUMERS) {
            const int a2 = t2 / G4, r2 = t2 - a2 * G4;
            if (a2 < nb) {
                const int g2 = r2 >> 2, p2 = r2 & 3;
                const double *src = wz + ((size_t)a2 * GN + g2 * N) * 4 + p2;
                double acc = 0.0;
                for (int mm = 0; mm < N; ++mm) acc += src[mm * 4];
                phiz[t2] = acc;
            }
        }
        if (!shfl_reduce) small_sync();
        for (int t2 = tid; t2 < rows; t2 += STP_CONSUMERS) {
            const int a2 = t2 / G4, r2 = t2 - a2 * G4, j2 = gb + a2;
            if (a2 < nb) {
                const double *Cp = base + lay.Ci + (size_t)a2 * G4 * G4 + r2;
                const double *pz = phiz + a2 * G4;
                double y = 0.0;
                for (int cc = 0; cc < G4; ++cc) y = fma(Cp[cc * G4], pz[cc], y);
                const double po = (GC > 0 && t2 == tid) ? phi_old : P.phi[(size_t)j2 * G4 + r2];
                ys[t2] = y;
                P.phi[(size_t)j2 * G4 + r2] = y;
                const double d = fabs(y - po);
                rmax = (d > rmax || !(d == d)) ? d : rmax;
            }
        }
        small_sync();
        for (int t2 = tid; t2 < rows; t2 += STP_CONSUMERS) {
            const int a2 = t2 / G4, r2 = t2 - a2 * G4, j2 = gb + a2;
            if (a2 < nb) {
                const int g2 = r2 >> 2, p2 = r2 & 3;
                const double *yy = ys + a2 * G4 + p2;
                double acc = 0.0;
                if (GC > 0 && t2 == tid) {
#pragma unroll
                    for (int gc = 0; gc < (GC > 0 ? GC : 1); ++gc) acc = fma(Kr[gc], yy[gc * 4], acc);
                    ss[t2] = dxq * 0.25 * acc;
                } else {
                    const double *Kp = S.transfer + ((size_t)j2 * G + g2) * G;
                    for (int gc = 0; gc < G; ++gc) acc = fma(Kp[gc], yy[gc * 4], acc);
                    ss[t2] = S.dx[j2] * 0.25 * acc;
                }
            }
        }
        consumer_sync();
        if (on) { // x = z + D^-1 U y
            const double *sv = ss + a * G4 + g * 4;
            const double s0 = sv[0], s1 = sv[1], s2 = sv[2], s3 = sv[3];
            double x[4];
#pragma unroll
            for (int p = 0; p < 4; ++p)
                x[p] = fma(Lent(p, 3), s3, fma(Lent(p, 2), s2, fma(Lent(p, 1), s1, fma(Lent(p, 0), s0, z[p]))));
            if (WANT_L2) {
                const double *old = base + lay.nb + (size_t)(a + 1) * n + gm * 4;
#pragma unroll
                for (int p = 0; p < 4; ++p) { const double d = x[p] - old[p]; l2 = fma(d, d, l2); }
            }
            double *out = P.psi_new + (size_t)j * n + gm * 4;
            *reinterpret_cast<double2 *>(out) = make_double2(x[0], x[1]);
            *reinterpret_cast<double2 *>(out + 2) = make_double2(x[2], x[3]);
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(&empty[st]); // this warp is done with the stage
        if (++st == stages) { st = 0; ph ^= 1; }
    }
    rmax = warp_max(rmax);
    if (lane == 0 && cell1 > cell0) atomicMax(P.resid_inf, resid_bits(rmax));
    if (WANT_L2) {
        l2 = warp_sum(l2);
        if (lane == 0 && cell1 > cell0) atomicAdd(P.resid_l2, l2);
    }
}

} // namespace

bool st_supported(const oci_ctx *ctx) { return 4 * ctx->G <= 32 && ctx->G * ctx->N <= ST_THREADS; }

// a1 + a2 of the structured path; returns the number of kernels launched
int launch_st_factor(oci_ctx *ctx)
{
    if (!st_supported(ctx)) return OCI_E_UNSUPPORTED;
    ProblemView P = make_view(ctx);
    OCI_CUDA_TRY(ctx, cudaMemsetAsync(ctx->info, 0x7f, sizeof(int), ctx->stream));
    const size_t total = (size_t)ctx->J * ctx->G * ctx->N;
    const bool pow2 = ctx->N <= 32 && (ctx->N & (ctx->N - 1)) == 0;
    int launches = 0;
    if (pow2 && ctx->opt_st_fused_setup != 0) {
        size_t gf = (total + 255) / 256;
        if (gf > (size_t)ctx->num_sms * 16) gf = (size_t)ctx->num_sms * 16;
        if (ctx->G == 1) {
            st_setup_fused_kernel<true><<<(int)gf, 256, 0, ctx->stream>>>(P, ctx->st_LinvT, ctx->st_Wg, ctx->st_Cinv, ctx->info);
            OCI_CUDA_TRY(ctx, cudaGetLastError());
            return 1;
        }
        st_setup_fused_kernel<false><<<(int)gf, 256, 0, ctx->stream>>>(P, ctx->st_LinvT, ctx->st_Wg, ctx->st_Cinv, ctx->info);
        OCI_CUDA_TRY(ctx, cudaGetLastError());
        launches = 1;
    } else {
        size_t g1 = (total + 127) / 128;
        if (g1 > (size_t)ctx->num_sms * 32) g1 = (size_t)ctx->num_sms * 32;
        st_setup_kernel<<<(int)g1, 128, 0, ctx->stream>>>(P, ctx->st_LinvT);
        OCI_CUDA_TRY(ctx, cudaGetLastError());
        size_t g3 = ((size_t)ctx->J * ctx->G * 16 + 255) / 256;
        if (g3 > (size_t)ctx->num_sms * 16) g3 = (size_t)ctx->num_sms * 16;
        st_wsum_kernel<<<(int)g3, 256, 0, ctx->stream>>>(P, ctx->st_LinvT, ctx->st_Wg);
        OCI_CUDA_TRY(ctx, cudaGetLastError());
        launches = 2;
    }
    size_t g2 = ((size_t)ctx->J + CAP_WARPS - 1) / CAP_WARPS;
    if (g2 > (size_t)ctx->num_sms * 4) g2 = (size_t)ctx->num_sms * 4;
    st_cap_kernel<<<(int)g2, CAP_WARPS * 32, 0, ctx->stream>>>(P, ctx->st_Wg, ctx->st_Cinv, ctx->info);
    OCI_CUDA_TRY(ctx, cudaGetLastError());
    return launches + 1;
}

int launch_st_iteration(oci_ctx *ctx, const IterParams &P, bool want_l2)
{
    StParams S;
    S.LinvT = ctx->st_LinvT; S.Cinv = ctx->st_Cinv; S.dx = ctx->dx; S.transfer = ctx->transfer;
    const int GN = ctx->G * ctx->N, G4 = 4 * ctx->G;
    if (ctx->opt_iterate_kernel == 1 && ctx->opt_ordering == 0) { // persistent bulk-copy pipeline (Jacobi ordering);
                                                                  // falls through when the ring would not fit
        // 256 consumer threads and two CTAs per SM; 128 and four when a cell takes a whole warp (measured: config 3,
        // G N = 32, 16.5 -> 13.4 us per iteration; config 5, G N = 16, is faster with 256: 45 against 47 us)
        const int CT = ctx->opt_st_ct == 128 || ctx->opt_st_ct == 256
                           ? ctx->opt_st_ct
                           : ((GN > 16 && GN <= 32 && ctx->opt_ctas_per_sm != 2) ? 128 : 256);
        const int CPB = CT / GN;
        const int max_ctas = CT == 128 ? 4 : 2;
        const StStage lay = st_stage_layout(ctx->N, ctx->G, CT);
        const size_t fixed = (size_t)2 * STP_MAX_STAGES * 8 + sizeof(double) * ((size_t)2 * ctx->N + (size_t)CPB * GN * 4 +
                                                                               (size_t)3 * CPB * G4 + (size_t)4 * GN) + 256;
        // two CTAs per SM by default: each is a lock-step sequence of short latency-bound phases, two of them overlap
        int ctas = ctx->opt_ctas_per_sm > 0 ? ctx->opt_ctas_per_sm : max_ctas;
        if (ctas > max_ctas) ctas = max_ctas;
        int stages = 0;
        for (; ctas >= 1; --ctas) {
            const size_t budget = ((size_t)ctx->max_smem_optin + 1024) / ctas - 1024; // 228 KB per SM, 1 KB reserved per CTA
            stages = budget > fixed ? (int)((budget - fixed) / ((size_t)lay.doubles * 8)) : 0;
            if (stages >= 2) break;
        }
        if (ctas < 1) ctas = 1;
        if (stages > STP_MAX_STAGES) stages = STP_MAX_STAGES;
        if (ctx->opt_stages > 0 && ctx->opt_stages < stages) stages = ctx->opt_stages;
        if (stages >= 2) {
            // every exchange of a batch inside one warp: N a power of two >= 4, a cell's G N threads do not straddle warps
            const int warp_local = (ctx->opt_st_warp_local != 0 && (ctx->G == 1 || ctx->G == 2 || ctx->G == 4 || ctx->G == 8) &&
                                    ctx->N >= 4 && (ctx->N & (ctx->N - 1)) == 0 && GN <= 32) ? 1 : 0;
            const size_t smem = fixed + (size_t)stages * lay.doubles * 8;
            int grid = ctx->num_sms * ctas;
            if (grid > (ctx->J + CPB - 1) / CPB) grid = (ctx->J + CPB - 1) / CPB;
#define OCI_STP_LAUNCH(L2_, GC_, CT_)                                                                              \
    do {                                                                                                           \
        OCI_CUDA_TRY(ctx, grant_smem(ctx, SLOT_STP + (((GC_ == 0 ? 0 : (GC_ == 1 ? 1 : (GC_ == 2 ? 2 : (GC_ == 4 ? 3 : 4)))) * 2 + \
                                                      (CT_ == 128 ? 0 : 1)) * 2 + (L2_ ? 1 : 0)),                  \
                                     (const void *)st_iterate_pipe_kernel<L2_, GC_, CT_>, smem));                  \
        OCI_CUDA_TRY(ctx, launch_pdl(st_iterate_pipe_kernel<L2_, GC_, CT_>, dim3(grid), dim3(CT_ + 32), smem,      \
                                     ctx->stream, P, S, stages, warp_local));                                    \
    } while (0)
#define OCI_STP_G(GC_)                                                                                             \
    do {                                                                                                           \
        if (CT == 128) {                                                                                           \
            if (want_l2) OCI_STP_LAUNCH(true, GC_, 128);                                                           \
            else OCI_STP_LAUNCH(false, GC_, 128);                                                                  \
        } else {                                                                                                   \
            if (want_l2) OCI_STP_LAUNCH(true, GC_, 256);                                                           \
            else OCI_STP_LAUNCH(false, GC_, 256);                                                                  \
        }                                                                                                          \
    } while (0)
            switch (ctx->G) {
            case 1: OCI_STP_G(1); break;
            case 2: OCI_STP_G(2); break;
            case 4: OCI_STP_G(4); break;
            case 8: OCI_STP_G(8); break;
            default: OCI_STP_G(0); break;
            }
#undef OCI_STP_G
#undef OCI_STP_LAUNCH
            OCI_CUDA_TRY(ctx, cudaGetLastError());
            return 1;
        }
    }
    const int CPB = ST_THREADS / GN;
    const size_t smem = sizeof(double) * ((size_t)2 * ctx->N + (size_t)CPB * GN * 4 + (size_t)3 * CPB * G4);
#define OCI_ST_LAUNCH(GC_)                                                                                         \
    do {                                                                                                           \
        if (want_l2) st_iterate_kernel<true, GC_><<<grid, ST_THREADS, smem, ctx->stream>>>(Q, S);                  \
        else st_iterate_kernel<false, GC_><<<grid, ST_THREADS, smem, ctx->stream>>>(Q, S);                         \
    } while (0)
    // ordering 1 (red-black): the even cells, then the odd cells, in place on the current iterate
    const int ncolors = ctx->opt_ordering == 1 ? 2 : 1;
    for (int color = 0; color < ncolors; ++color) {
        IterParams Q = P;
        Q.color = color;
        Q.ncolors = ncolors;
        if (ncolors == 2) Q.psi_new = const_cast<double *>(P.psi_old);
        const int Jc = (ctx->J - color + ncolors - 1) / ncolors;
        if (Jc < 1) continue;
        const int grid = (Jc + CPB - 1) / CPB; // one batch of CPB cells per CTA: CTA turnover hides the load latency
        switch (ctx->G) {
        case 1: OCI_ST_LAUNCH(1); break;
        case 2: OCI_ST_LAUNCH(2); break;
        case 4: OCI_ST_LAUNCH(4); break;
        case 8: OCI_ST_LAUNCH(8); break;
        default: OCI_ST_LAUNCH(0); break;
        }
    }
#undef OCI_ST_LAUNCH
    OCI_CUDA_TRY(ctx, cudaGetLastError());
    return ncolors;
}

// f2: k iterations in one cooperative launch. Applies (auto) to small problems (<= 8 MB per iteration), where the fixed
// cost of a launch is what an iteration costs (measured: config 1 5.6 -> 3.9 us, config 2 6.2 -> 5.1 us per iteration;
// from ~10 MB on the pipelined per-iteration kernel is faster); "persistent" = 1 forces it, 0 disables it.
int launch_st_multi(oci_ctx *ctx, int slot0, int k, bool want_l2, bool check_between)
{
    if (ctx->opt_solve_mode != 1 || ctx->opt_persistent == 0 || ctx->opt_ordering != 0 || k < 2) return 0;
    const int GN = ctx->G * ctx->N, CPB = ST_THREADS / GN, G4 = 4 * ctx->G;
    const size_t bytes_per_iter = (size_t)ctx->J * (36 * (size_t)ctx->n + 136 * (size_t)ctx->G * ctx->G + 64 * ctx->G + 8);
    if (ctx->opt_persistent < 0 && bytes_per_iter > ((size_t)8 << 20)) return 0;
    int coop = 0;
    if (cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, ctx->device) != cudaSuccess || !coop) return 0;
    const size_t smem = sizeof(double) * ((size_t)2 * ctx->N + (size_t)CPB * GN * 4 + (size_t)3 * CPB * G4);
    IterParams P;
    P.stop = make_stop(ctx, slot0, false);
    P.J = ctx->J; P.N = ctx->N; P.G = ctx->G; P.n = ctx->n;
    P.bc_left = ctx->bc_left; P.bc_right = ctx->bc_right;
    P.Minv = nullptr; P.c = ctx->c;
    P.psi_old = ctx->psi[ctx->cur]; P.psi_new = ctx->psi[ctx->cur ^ 1];
    P.phi = ctx->phi; P.mu = ctx->mu; P.w = ctx->w;
    P.inc_left = ctx->inc_left; P.inc_right = ctx->inc_right;
    P.resid_inf = ctx->resid_inf + slot0; P.resid_l2 = ctx->resid_l2 + slot0;
    P.cpb = 1; P.S = 1; P.cw = ctx->n; P.nch = 1; P.n_items = ctx->J; P.stages = 0; P.chunk_doubles = 0;
    P.color = 0; P.ncolors = 1; P.reverse = 0;
    StParams S;
    S.LinvT = ctx->st_LinvT; S.Cinv = ctx->st_Cinv; S.dx = ctx->dx; S.transfer = ctx->transfer;
    StMulti M;
    M.n_iters = k; M.slot0 = slot0; M.check_between = check_between ? 1 : 0; M.rule = ctx->stop_rule; M.tol = ctx->stop_tol;
    M.resid_inf = ctx->resid_inf; M.resid_l2 = ctx->resid_l2; M.executed = ctx->ctrl;
    void *args[] = {&P, &S, &M};
    const void *fn = nullptr;
#define OCI_STM_PICK(GC_) fn = want_l2 ? (const void *)st_iterate_multi_kernel<true, GC_> : (const void *)st_iterate_multi_kernel<false, GC_>
    switch (ctx->G) {
    case 1: OCI_STM_PICK(1); break;
    case 2: OCI_STM_PICK(2); break;
    case 4: OCI_STM_PICK(4); break;
    case 8: OCI_STM_PICK(8); break;
    default: OCI_STM_PICK(0); break;
    }
#undef OCI_STM_PICK
    int per_sm = 0;
    OCI_CUDA_TRY(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, fn, ST_THREADS, smem));
    if (per_sm < 1) return 0;
    int grid = (ctx->J + CPB - 1) / CPB;
    if (grid > per_sm * ctx->num_sms) grid = per_sm * ctx->num_sms; // all CTAs co-resident: the grid barrier needs it
    OCI_CUDA_TRY(ctx, cudaLaunchCooperativeKernel(fn, dim3(grid), dim3(ST_THREADS), args, smem, ctx->stream));
    if (k & 1) ctx->cur ^= 1; // as k single launches would have left it
    return 1;
}
