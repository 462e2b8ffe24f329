// factor.cu -- a1 (assemble A_j) + a2 (eliminate with partial pivoting) of SURVEY.md section 8(a).
//
// A_j = [delta_gg' L_{c,j,g} - S_{g'->g,j}]  (Eq. 40b), L_c block-diagonal in the ordinate
// (Eq. 8a-b), S_{(g,m,p),(g',m',p')} = delta_pp' (dx_j K_j[g][g'] / 4) w_m'  (Eq. 10 / 39,
// PAPER.md:154, 320, read as DESIGN.md A2). The matrix is assembled straight into on-chip memory and never
// written to HBM un-eliminated. Elimination is Gaussian elimination with partial (row) pivoting -- the same
// pivots `_gesv` takes in Alg. 2 -- carried through to the inverse (Gauss-Jordan, in
// place, implicit row exchange), because the iterate kernel streams A_j^{-1}.
#include "common.cuh"
#include <limits.h>

namespace {

constexpr int FACTOR_THREADS = 256;

// Entry (i, c) of A_j, every rounding explicit (bit-identical to an uncontracted evaluation).
__device__ __forceinline__ double a_entry(const ProblemView &P, int cell, int i, int c)
{
    const int N = P.N, G = P.G;
    const int p = i & 3, bm = i >> 2, m = bm % N, g = bm / N;
    const int pp = c & 3, bmc = c >> 2, mc = bmc % N, gc = bmc / N;
    const double dx = P.dx[cell];
    double val = 0.0;
    if (bm == bmc) val = lc_entry(p, pp, dx, P.sigma_t[(size_t)cell * G + g], P.v[g], P.dt, P.mu[m]);
    if (p == pp) {
        const double K = P.transfer[((size_t)cell * G + g) * G + gc];
        const double s = __dmul_rn(__dmul_rn(__dmul_rn(dx, K), 0.25), P.w[mc]); // dx K / 4 * w_m'
        val = __dsub_rn(val, s);
    }
    return val;
}

// One CTA per cell (grid-stride). W is the n x n working array, row-major with leading dimension ldw:
// in shared memory when it fits (ldw = n + 1, conflict-free column access), else in a per-CTA global scratch
// that stays L2-resident.
template <bool GLOBAL_W>
__global__ void __launch_bounds__(FACTOR_THREADS)
factor_gj_kernel(ProblemView P, double *__restrict__ Minv, double *__restrict__ scratch, int ldw, int *info)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int n = P.n;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    constexpr int NW = FACTOR_THREADS / 32;

    double *sm = reinterpret_cast<double *>(smem_raw);
    double *colk = sm;               // [n]
    double *prow = colk + n;         // [n]
    double *wmax = prow + n;         // [NW]
    int *widx = reinterpret_cast<int *>(wmax + NW); // [NW]
    int *rho = widx + NW;            // [n] pivot row of step k
    int *rhoinv = rho + n;           // [n]
    int *used = rhoinv + n;          // [n]
    double *Wsm = reinterpret_cast<double *>(used + n + ((n + NW) & 1)); // keep 8-byte alignment
    double *W = GLOBAL_W ? scratch + (size_t)blockIdx.x * n * ldw : Wsm;

    for (int cell = blockIdx.x; cell < P.J; cell += gridDim.x) {
        // ---- a1: assemble
        for (int i = warp; i < n; i += NW)
            for (int c = lane; c < n; c += 32) W[(size_t)i * ldw + c] = a_entry(P, cell, i, c);
        for (int i = tid; i < n; i += FACTOR_THREADS) used[i] = 0;
        __syncthreads();

        bool singular = false;
        // ---- a2: elimination, step k eliminates column k with the pivot row rho_k
        for (int k = 0; k < n; ++k) {
            double cand = -1.0;
            int ci = INT_MAX;
            for (int i = tid; i < n; i += FACTOR_THREADS) {
                const double vv = W[(size_t)i * ldw + k];
                colk[i] = vv;
                const double a = used[i] ? -1.0 : fabs(vv);
                if (a > cand) { cand = a; ci = i; }
            }
            // arg-max by warp shuffles: larger |entry| wins, ties go to the lower row
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
                const double oc = __shfl_xor_sync(0xffffffffu, cand, o);
                const int oi = __shfl_xor_sync(0xffffffffu, ci, o);
                if (oc > cand || (oc == cand && oi < ci)) { cand = oc; ci = oi; }
            }
            if (lane == 0) { wmax[warp] = cand; widx[warp] = ci; }
            __syncthreads();
            double best = wmax[0];
            int r = widx[0];
#pragma unroll
            for (int q = 1; q < NW; ++q) {
                const double oc = wmax[q];
                const int oi = widx[q];
                if (oc > best || (oc == best && oi < r)) { best = oc; r = oi; }
            }
            if (!(best > 0.0)) { singular = true; break; } // uniform across the CTA
            const double inv = 1.0 / colk[r];
            for (int c = tid; c < n; c += FACTOR_THREADS)
                prow[c] = (c == k ? 1.0 : W[(size_t)r * ldw + c]) * inv;
            if (tid == 0) { used[r] = 1; rho[k] = r; rhoinv[r] = k; }
            __syncthreads();
            for (int i = warp; i < n; i += NW) {
                double *Wi = W + (size_t)i * ldw;
                if (i == r) {
                    for (int c = lane; c < n; c += 32) Wi[c] = prow[c];
                } else {
                    const double f = colk[i];
                    if (f != 0.0)
                        for (int c = lane; c < n; c += 32) {
                            const double base = (c == k) ? 0.0 : Wi[c];
                            Wi[c] = fma(-f, prow[c], base);
                        }
                }
            }
            __syncthreads();
        }
        if (singular) {
            if (tid == 0) atomicMin(info, cell + 1);
            // leave a NaN-free but meaningless block behind: zero it
            for (int e = tid; e < n * n; e += FACTOR_THREADS) Minv[(size_t)cell * n * n + e] = 0.0;
            __syncthreads();
            continue;
        }
        // ---- store A^{-1} column-major: Ainv[kappa][rho_j] = W[rho_kappa][j]  (un-scrambles the implicit exchange)
        double *out = Minv + (size_t)cell * n * n;
        for (int j = warp; j < n; j += NW) {
            const int col = rho[j];
            for (int i = lane; i < n; i += 32) out[(size_t)col * n + rhoinv[i]] = W[(size_t)i * ldw + j];
        }
        __syncthreads();
    }
}

__global__ void assemble_one_kernel(ProblemView P, int cell, double *__restrict__ A)
{
    const int n = P.n;
    for (int e = blockIdx.x * blockDim.x + threadIdx.x; e < n * n; e += gridDim.x * blockDim.x)
        A[e] = a_entry(P, cell, e / n, e % n);
}

size_t factor_smem_bytes(int n, bool global_w)
{
    constexpr int NW = FACTOR_THREADS / 32;
    size_t b = (size_t)(2 * n + NW) * sizeof(double) + (size_t)(NW + 3 * n + 1) * sizeof(int);
    b = (b + 15) & ~(size_t)15;
    if (!global_w) b += (size_t)n * (n + 1) * sizeof(double);
    return b;
}

} // namespace

// Scratch the factor path may need: per-CTA n x n working arrays when n is too large for shared memory,
// and at least one n x n matrix for the debug getters.
size_t factor_scratch_bytes(int n, int num_sms, int max_smem_optin)
{
    size_t one = (size_t)n * n * sizeof(double);
    if (factor_smem_bytes(n, false) <= (size_t)max_smem_optin) return one;
    return one * (size_t)num_sms * 4;
}

int launch_factor(oci_ctx *ctx)
{
    const int n = ctx->n;
    ProblemView P = make_view(ctx);
    OCI_CUDA_TRY(ctx, cudaMemsetAsync(ctx->info, 0x7f, sizeof(int), ctx->stream)); // 0x7f7f7f7f = "none"
    const bool global_w = factor_smem_bytes(n, false) > (size_t)ctx->max_smem_optin;
    const size_t smem = factor_smem_bytes(n, global_w);
    int grid;
    if (!global_w) {
        OCI_CUDA_TRY(ctx, cudaFuncSetAttribute(factor_gj_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                               (int)smem));
        int per_sm = 1;
        OCI_CUDA_TRY(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, factor_gj_kernel<false>,
                                                                        FACTOR_THREADS, smem));
        if (per_sm < 1) per_sm = 1;
        grid = ctx->num_sms * per_sm;
        if (grid > ctx->J) grid = ctx->J;
        factor_gj_kernel<false><<<grid, FACTOR_THREADS, smem, ctx->stream>>>(P, ctx->Minv, nullptr, n + 1, ctx->info);
    } else {
        grid = ctx->num_sms * 4;
        if (grid > ctx->J) grid = ctx->J;
        if ((size_t)grid * n * n * sizeof(double) > ctx->scratch_bytes) return OCI_E_WORKSPACE;
        factor_gj_kernel<true><<<grid, FACTOR_THREADS, smem, ctx->stream>>>(P, ctx->Minv, ctx->scratch, n, ctx->info);
    }
    OCI_CUDA_TRY(ctx, cudaGetLastError());
    return 1;
}

int launch_assemble_one(oci_ctx *ctx, int cell, double *A_dev_rowmajor)
{
    ProblemView P = make_view(ctx);
    assemble_one_kernel<<<32, 256, 0, ctx->stream>>>(P, cell, A_dev_rowmajor);
    OCI_CUDA_TRY(ctx, cudaGetLastError());
    return 1;
}
