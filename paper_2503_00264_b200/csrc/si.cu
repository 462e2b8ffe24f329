// si.cu -- a9..a11 of SURVEY.md section 8(a): the source-iteration comparator (Alg. 1, PAPER.md:366-411;
// Appendix A, Eq. 42-46), "parallel over angles x groups and serial in space".
//
// One source iteration:
//   s_{j,g,p} = sum_g' K_j[g][g'] phi^(l)_{j,g',p}                       (all groups lagged, A5/A13)
//   for every (g,m), cells in the direction of mu_m:   L_{c,j,g,m} psi = d + mu * (upstream psi of THIS sweep)
//   phi^(l+1) = sum_m w_m psi_m,  r = max |phi^(l+1) - phi^(l)|
// The 4x4 solve of Eq. 42 is linear in the incident edge flux, and only the two "outgoing" unknowns feed the
// next cell (Eq. 5a-b). The work is therefore split into
//   si_source : (parallel over j,g,m)  base = L^-1 d            -- everything that does not depend on the sweep
//   si_sweep  : (parallel over g,m; SERIAL over j)  in_{j+1} = base_out_j + T_j in_j   (2x2 affine map per cell)
//   si_finish : (parallel over j,g,m)  psi = base + C in,  phi, residual
// which is the same arithmetic as solving cell after cell, re-associated; the serial chain per cell is two
// dependent fused multiply-adds instead of a 4x4 solve.
#include "common.cuh"

namespace {

// ---- 4x4 inverse by Gauss-Jordan with partial pivoting, fully unrolled (registers only) ---------------------
__device__ __forceinline__ void inv4(double (&a)[4][4], double (&b)[4][4])
{
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) b[i][j] = (i == j) ? 1.0 : 0.0;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        int p = k;
        double best = fabs(a[k][k]);
#pragma unroll
        for (int i = k + 1; i < 4; ++i) {
            const double t = fabs(a[i][k]);
            if (t > best) { best = t; p = i; }
        }
#pragma unroll
        for (int i = k + 1; i < 4; ++i)
            if (p == i) {
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    double t = a[k][j]; a[k][j] = a[i][j]; a[i][j] = t;
                    t = b[k][j]; b[k][j] = b[i][j]; b[i][j] = t;
                }
            }
        const double inv = 1.0 / a[k][k];
#pragma unroll
        for (int j = 0; j < 4; ++j) { a[k][j] *= inv; b[k][j] *= inv; }
#pragma unroll
        for (int i = 0; i < 4; ++i)
            if (i != k) {
                const double f = a[i][k];
#pragma unroll
                for (int j = 0; j < 4; ++j) { a[i][j] = fma(-f, a[k][j], a[i][j]); b[i][j] = fma(-f, b[k][j], b[i][j]); }
            }
    }
}

// Once per (problem, dt): Linv[j][g][m][4][4] = L_{c,j,g,m}^{-1} (Eq. 8b / 42) and
// C[j][g][m][p][lev] = |mu_m| Linv[p][row that receives the incident flux of level lev].
__global__ void si_setup_kernel(ProblemView P, double *__restrict__ Linv, double *__restrict__ C)
{
    const size_t total = (size_t)P.J * P.G * P.N;
    for (size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x; e < total; e += (size_t)gridDim.x * blockDim.x) {
        const int m = (int)(e % P.N);
        const size_t jg = e / P.N;
        const int g = (int)(jg % P.G);
        const size_t j = jg / P.G;
        const double mu = P.mu[m];
        double a[4][4], b[4][4];
#pragma unroll
        for (int p = 0; p < 4; ++p)
#pragma unroll
            for (int pp = 0; pp < 4; ++pp) a[p][pp] = lc_entry(p, pp, P.dx[j], P.sigma_t[jg], P.v[g], P.dt, mu);
        inv4(a, b);
        double *Lo = Linv + e * 16;
#pragma unroll
        for (int p = 0; p < 4; ++p)
#pragma unroll
            for (int pp = 0; pp < 4; ++pp) Lo[p * 4 + pp] = b[p][pp];
        const double am = fabs(mu);
        double *Co = C + e * 8;
#pragma unroll
        for (int p = 0; p < 4; ++p) {
            // mu > 0: rows (k,L)=0 and (k+1/2,L)=2 receive the incident flux; mu < 0: rows 1 and 3 (Eq. 43b-c)
            Co[p * 2 + 0] = am * (mu > 0.0 ? b[p][0] : b[p][1]);
            Co[p * 2 + 1] = am * (mu > 0.0 ? b[p][2] : b[p][3]);
        }
    }
}

// a9: d_{j,g,m} (Eq. 43b-c, without the incident term) and base = Linv d.
__global__ void si_source_kernel(StopCheck stop, ProblemView P, const double *__restrict__ q,
                                 const double *__restrict__ psi_prev, const double *__restrict__ phi,
                                 const double *__restrict__ Linv, double *__restrict__ base)
{
    if (stop_reached(stop)) return;
    const size_t total = (size_t)P.J * P.G * P.N;
    for (size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x; e < total; e += (size_t)gridDim.x * blockDim.x) {
        const size_t jg = e / P.N;
        const int g = (int)(jg % P.G);
        const size_t j = jg / P.G;
        const double dx = P.dx[j];
        const double *Kj = P.transfer + (j * P.G + g) * P.G;
        const double *phij = phi + j * P.G * 4;
        double d[4];
#pragma unroll
        for (int p = 0; p < 4; ++p) {
            double s = 0.0;
            for (int gp = 0; gp < P.G; ++gp) s = fma(Kj[gp], phij[gp * 4 + p], s);
            d[p] = dx * 0.25 * (s + q[jg * 4 + p]);
        }
        const double half_gam = dx / (2.0 * P.v[g] * P.dt);
        d[0] = fma(half_gam, psi_prev[e * 2 + 0], d[0]);
        d[1] = fma(half_gam, psi_prev[e * 2 + 1], d[1]);
        const double *L = Linv + e * 16;
#pragma unroll
        for (int p = 0; p < 4; ++p)
            base[e * 4 + p] = fma(L[p * 4 + 3], d[3], fma(L[p * 4 + 2], d[2], fma(L[p * 4 + 1], d[1], L[p * 4 + 0] * d[0])));
    }
}

// a10: the sweep. One warp per CTA sweeps LPC ordinates (g,m): all 32 lanes stage the per-cell 2x2 maps and
// base values of the next cells into a shared-memory ring with cp.async (the loads do not depend on the
// chain), the first LPC lanes run the serial chain out of shared memory.
constexpr int LPC = 4;
constexpr int TC = 32;
constexpr int SW_STAGES = 4;

__global__ void __launch_bounds__(32) si_sweep_kernel(StopCheck stop, int J, int N, int G, int bc_left, int bc_right,
                                                      const double *__restrict__ mu, const double *__restrict__ C,
                                                      const double *__restrict__ base,
                                                      const double *__restrict__ psi_old,
                                                      const double *__restrict__ inc_left,
                                                      const double *__restrict__ inc_right, double *__restrict__ in_out)
{
    __shared__ __align__(16) double tile[SW_STAGES][TC][LPC][8]; // [C out0 (2)][C out1 (2)][base (4)]
    if (stop_reached(stop)) return;
    const int lane = threadIdx.x;
    const int GN = G * N, n = 4 * GN;
    const int gm0 = blockIdx.x * LPC;
    const int n_tiles = (J + TC - 1) / TC;

    auto stage_tile = [&](int t) {
        if (t < n_tiles) {
            double(*dst)[LPC][8] = tile[t % SW_STAGES];
            for (int idx = lane; idx < TC * LPC * 4; idx += 32) {
                const int part = idx & 3, l = (idx >> 2) % LPC, u = idx / (4 * LPC);
                const int gm = gm0 + l, jj = t * TC + u;
                if (gm < GN && jj < J) {
                    const bool fwd = mu[gm % N] > 0.0;
                    const size_t j = fwd ? jj : J - 1 - jj;
                    const size_t cell_gm = j * GN + gm;
                    const int o0 = fwd ? 1 : 0; // outgoing unknowns: (k,R),(k+1/2,R) for mu>0; (k,L),(k+1/2,L) for mu<0
                    const double *src = part == 0   ? C + cell_gm * 8 + o0 * 2
                                        : part == 1 ? C + cell_gm * 8 + (o0 + 2) * 2
                                        : part == 2 ? base + cell_gm * 4
                                                    : base + cell_gm * 4 + 2;
                    const uint32_t d = smem_u32(&dst[u][l][part * 2]);
                    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(d), "l"(src) : "memory");
                }
            }
        }
        asm volatile("cp.async.commit_group;" ::: "memory");
    };

    for (int t = 0; t < SW_STAGES - 1; ++t) stage_tile(t);

    const int gm = gm0 + lane;
    const bool active = lane < LPC && gm < GN;
    bool fwd = true;
    double in0 = 0.0, in1 = 0.0;
    if (active) {
        const int g = gm / N, m = gm % N;
        fwd = mu[m] > 0.0;
        const int bc = fwd ? bc_left : bc_right;
        if (bc == OCI_BC_REFLECTIVE) { // mirror ordinate of the boundary cell, from iteration l (A12)
            const double *cellp = psi_old + (fwd ? (size_t)0 : (size_t)(J - 1) * n) + (size_t)(g * N + (N - 1 - m)) * 4;
            in0 = cellp[fwd ? 0 : 1];
            in1 = cellp[fwd ? 2 : 3];
        } else if (bc == OCI_BC_PRESCRIBED) {
            const double *ip = (fwd ? inc_left : inc_right) + (size_t)gm * 2;
            in0 = ip[0];
            in1 = ip[1];
        }
    }

    for (int t = 0; t < n_tiles; ++t) {
        stage_tile(t + SW_STAGES - 1);
        asm volatile("cp.async.wait_group %0;" ::"n"(SW_STAGES - 1) : "memory");
        __syncwarp();
        if (active) {
            const double(*src)[LPC][8] = tile[t % SW_STAGES];
            const int cells = min(TC, J - t * TC);
#pragma unroll 8
            for (int u = 0; u < cells; ++u) {
                const double *s = src[u][lane];
                const int jj = t * TC + u;
                const size_t j = fwd ? jj : J - 1 - jj;
                *reinterpret_cast<double2 *>(in_out + (j * GN + gm) * 2) = make_double2(in0, in1);
                const int ob = fwd ? 1 : 0;
                const double o0 = fma(s[0], in0, fma(s[1], in1, s[4 + ob]));
                const double o1 = fma(s[2], in0, fma(s[3], in1, s[4 + ob + 2]));
                in0 = o0;
                in1 = o1;
            }
        }
        __syncwarp();
    }
}

// a11 (+ the rest of a10): psi = base + C in for every (j,g,m); phi = sum_m w_m psi_m; residual.
constexpr int FIN_THREADS = 256;
template <bool WANT_L2>
__global__ void __launch_bounds__(FIN_THREADS)
si_finish_kernel(StopCheck stop, int J, int N, int G, const double *__restrict__ w, const double *__restrict__ C,
                 const double *__restrict__ base, const double *__restrict__ in_, double *__restrict__ psi,
                 double *__restrict__ phi, unsigned long long *resid_inf, double *resid_l2)
{
    __shared__ double ws[FIN_THREADS][4];
    if (stop_reached(stop)) return;
    if (blockIdx.x == 0 && threadIdx.x == 0) *stop.executed = stop.slot + 1;
    const int pairs_per_block = FIN_THREADS / N; // (j,g) pairs per block
    const size_t n_pairs = (size_t)J * G;
    const int tid = threadIdx.x, lane = tid & 31;
    double rmax = 0.0, l2 = 0.0;
    for (size_t pair0 = (size_t)blockIdx.x * pairs_per_block; pair0 < n_pairs; pair0 += (size_t)gridDim.x * pairs_per_block) {
        const int local_pair = tid / N, m = tid - local_pair * N;
        const size_t pair = pair0 + local_pair;
        __syncthreads();
        if (local_pair < pairs_per_block && pair < n_pairs) {
            const size_t e = pair * N + m;
            const double i0 = in_[e * 2], i1 = in_[e * 2 + 1];
            const double wm = w[m];
#pragma unroll
            for (int p = 0; p < 4; ++p) {
                const double x = fma(C[e * 8 + p * 2], i0, fma(C[e * 8 + p * 2 + 1], i1, base[e * 4 + p]));
                psi[e * 4 + p] = x;
                ws[tid][p] = wm * x;
            }
        }
        __syncthreads();
        const int lp = tid >> 2, p = tid & 3;
        if (lp < pairs_per_block && pair0 + lp < n_pairs) {
            double s = 0.0;
            for (int mm = 0; mm < N; ++mm) s += ws[lp * N + mm][p];
            const size_t o = (pair0 + lp) * 4 + p;
            const double d = s - phi[o];
            phi[o] = s;
            const double ad = fabs(d);
            rmax = (ad > rmax || !(ad == ad)) ? ad : rmax;
            if (WANT_L2) l2 = fma(d, d, l2);
        }
    }
    rmax = warp_max(rmax);
    if (lane == 0) atomicMax(resid_inf, resid_bits(rmax));
    if (WANT_L2) {
        l2 = warp_sum(l2);
        if (lane == 0) atomicAdd(resid_l2, l2);
    }
}

inline int grid_for(size_t total, int threads, int num_sms)
{
    size_t g = (total + threads - 1) / threads;
    size_t cap = (size_t)num_sms * 16;
    if (g > cap) g = cap;
    if (g < 1) g = 1;
    return (int)g;
}

} // namespace

int launch_si_setup(oci_ctx *ctx)
{
    ProblemView P = make_view(ctx);
    const size_t total = (size_t)ctx->J * ctx->G * ctx->N;
    si_setup_kernel<<<grid_for(total, 128, ctx->num_sms), 128, 0, ctx->stream>>>(P, ctx->si_Linv, ctx->si_T);
    OCI_CUDA_TRY(ctx, cudaGetLastError());
    return 1;
}

int launch_si_iteration(oci_ctx *ctx, int hist_slot, bool want_l2, bool check_prev)
{
    ProblemView P = make_view(ctx);
    const StopCheck stop = make_stop(ctx, hist_slot, check_prev);
    const int GN = ctx->G * ctx->N;
    const size_t total = (size_t)ctx->J * GN;
    double *psi = ctx->psi[ctx->cur];
    si_source_kernel<<<grid_for(total, 256, ctx->num_sms), 256, 0, ctx->stream>>>(stop, P, ctx->q, ctx->psi_prev, ctx->phi,
                                                                                   ctx->si_Linv, ctx->si_base);
    OCI_CUDA_TRY(ctx, cudaGetLastError());
    si_sweep_kernel<<<(GN + LPC - 1) / LPC, 32, 0, ctx->stream>>>(stop, ctx->J, ctx->N, ctx->G, ctx->bc_left, ctx->bc_right,
                                                                  ctx->mu, ctx->si_T, ctx->si_base, psi, ctx->inc_left,
                                                                  ctx->inc_right, ctx->si_in);
    OCI_CUDA_TRY(ctx, cudaGetLastError());
    const int pairs_per_block = FIN_THREADS / ctx->N;
    size_t blocks = ((size_t)ctx->J * ctx->G + pairs_per_block - 1) / pairs_per_block;
    if (blocks > (size_t)ctx->num_sms * 16) blocks = (size_t)ctx->num_sms * 16;
    if (want_l2)
        si_finish_kernel<true><<<(int)blocks, FIN_THREADS, 0, ctx->stream>>>(stop, ctx->J, ctx->N, ctx->G, ctx->w, ctx->si_T,
                                                                            ctx->si_base, ctx->si_in, psi, ctx->phi,
                                                                            ctx->resid_inf + hist_slot,
                                                                            ctx->resid_l2 + hist_slot);
    else
        si_finish_kernel<false><<<(int)blocks, FIN_THREADS, 0, ctx->stream>>>(stop, ctx->J, ctx->N, ctx->G, ctx->w, ctx->si_T,
                                                                             ctx->si_base, ctx->si_in, psi, ctx->phi,
                                                                             ctx->resid_inf + hist_slot,
                                                                             ctx->resid_l2 + hist_slot);
    OCI_CUDA_TRY(ctx, cudaGetLastError());
    return 3;
}
