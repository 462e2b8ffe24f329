// common.cuh -- context, launch-parameter structs and small device helpers shared by the kernels of
// liboci_b200.so. Nothing here is shared with oracle/ (see DESIGN.md "Independence").
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stddef.h>
#include "../../include/oci.h"

#define OCI_CUDA_TRY(ctx, expr)                                   \
    do {                                                          \
        cudaError_t _e = (expr);                                  \
        if (_e != cudaSuccess) {                                  \
            (ctx)->last_cuda = (int)_e;                           \
            return OCI_E_CUDA;                                    \
        }                                                         \
    } while (0)

constexpr int OCI_SMEM_SLOTS = 48;
enum { // one slot per kernel instantiation that needs more than 48 KB of dynamic shared memory
    SLOT_WPC = 0,      // + 2 * (RPL index) + want_l2   (6 slots)
    SLOT_STREAM = 6,   // + want_l2                     (2 slots)
    SLOT_SWEEP = 8,    // + lanes index                 (3 slots)
    SLOT_STP = 11,     // + ((GC index) * 2 + CT index) * 2 + want_l2   (20 slots)
    SLOT_FACTOR = 32,  // factor kernels
    SLOT_RESIDENT = 40 // + want_l2 (2 slots)
};

// ------------------------------------------------------------------------------------------------------------
// Context. All device pointers are carved out of the caller's workspace (the library never cudaMallocs).
// ------------------------------------------------------------------------------------------------------------
struct oci_ctx {
    int J, N, G, n;
    double dt;
    int bc_left, bc_right;
    cudaStream_t stream;
    int device, num_sms, max_smem_optin;
    int last_cuda;

    // problem (device copies)
    double *dx, *sigma_t, *transfer, *v, *mu, *w;
    // per-step inputs / state
    double *q;          // [J][G][4]
    double *inc_left;   // [G][N][2]
    double *inc_right;  // [G][N][2]
    double *psi_prev;   // [J][G][N][2]   psi_{k-1/2}
    double *psi[2];     // [J][n]         Jacobi double buffer; psi[cur] is the current iterate
    int cur;
    double *phi;        // [J][G][4]      scalar flux of psi[cur]
    double *c;          // [J][n]         constant part of b_j (a3)
    // OCI factors
    double *Minv;       // [J][n(col)][n(row)]  A_j^{-1}, column-major per cell
    double *scratch;    // factor kernel scratch (n > smem capacity) / debug matrix
    size_t scratch_bytes;
    int *info;          // [1] singular-cell flag (min 1-based cell index, INT_MAX = none)
    // SI data
    double *si_Linv;    // [J][G][N][16]  inverse of L_{c,j,g,m} (Eq. 42)
    double *si_T;       // [J][G*N][4][2] C = |mu| Linv[:, incident rows]; its outgoing rows are the sweep's 2x2 map
    double *si_base;    // [J][G*N][4]    Linv * d (no incident term)
    double *si_in;      // [J][G*N][2]    incident edge flux of cell j found by the sweep
    double *si_T2sw;    // [ceil(GN/lpc)][J][lpc][2][2]  incident -> outgoing 2x2 map, sweep order (si.cu sweep_index)
    double *si_bsw;     // [ceil(GN/lpc)][J][lpc][2]     outgoing entries of si_base, sweep order
    double *si_scan;    // scan mode ("si_sweep" = 1): per-thread prefixes and per-block aggregates (si.cu)
    size_t si_scan_bytes;
    // structured cell solve ("solve_mode" = 1; structured.cu)
    double *st_LinvT;   // [J][8][G*N]    rows (k,L), (k+1/2,L) of L_{c,j,g,m}^-1, ordinate-fastest (structured.cu ST_LK)
    double *st_Wg;      // [J][G][16]     sum_m w_m L^-1_{j,g,m}
    double *st_Cinv;    // [J][4G(col)][4G(row)]  (I - V^T D^-1 U)^-1, column-major per cell
    // residual history (device) + pinned host mirror
    unsigned long long *resid_inf; // [OCI_RESID_CAP] bit pattern of a non-negative double
    double *resid_l2;              // [OCI_RESID_CAP] sum of squares
    double *h_resid;               // pinned host, 2 * OCI_RESID_CAP
    int hist_len;                  // iterations recorded since the history was last reset
    int hist_dirty;                // residual slots [0, hist_dirty) may have been written since they were last zeroed
    int hist_has_l2;

    int *ctrl;                     // [4] ctrl[0] = iterations of the current step that really ran (device-side stop)
    double stop_tol;               // stop rule the device applies between the iterations of one batch
    int stop_rule;

    bool factored, c_valid, si_valid, phi_valid;
    bool factor_flagged; // the last oci_factor reported singular cells: the other cells' inverses are in place (debug getter)
    // options
    int opt_iterate_kernel, opt_stages, opt_ctas_per_sm, opt_factor_kernel, opt_factor_update, opt_factor_cluster, opt_refactor_every_step, opt_si_lanes, opt_solve_mode, opt_si_sweep, opt_persistent, opt_ordering, opt_st_warp_local, opt_st_ct, opt_st_fused_setup;
    // largest dynamic shared-memory size already granted (cudaFuncSetAttribute) to each kernel this context launches;
    // kept per context (= per device), never in function-local statics
    size_t smem_granted[OCI_SMEM_SLOTS];
    // production factor kernel whose attributes are set and whose occupancy-derived grid is known (factor.cu): with
    // refactor_every_step the factor launch is on every step's critical path, so this host work is done once
    const void *factor_fn;
    int factor_grid;
    // timing
    cudaEvent_t ev0, ev1;
    cudaEvent_t evf0, evf1;        // bracket the factor launch (own pair: a step enqueues factor + iterations before it syncs)
    double last_ms[3];
    long long last_launches[3];
};

// ------------------------------------------------------------------------------------------------------------
// Kernel parameter blocks
// ------------------------------------------------------------------------------------------------------------
struct ProblemView {
    int J, N, G, n;
    double dt;
    int bc_left, bc_right;
    const double *dx, *sigma_t, *transfer, *v, *mu, *w;
};

// Device-side stop: iteration `slot` of a batch first looks at the residual slot - 1, which
// is complete because launches are stream-ordered, and returns at once if the stop rule held there. Skipped slots
// keep their memset value 0, which makes the skip sticky. prev_inf == nullptr: no check (first slot of a batch,
// bare oci_iterate / si_iterate calls).
struct StopCheck {
    const unsigned long long *prev_inf; // resid_inf[slot - 1]
    const double *prev_l2;              // resid_l2[slot - 1]
    const double *prev2_l2;             // resid_l2[slot - 2], nullptr if slot - 1 == 0 (Eq. 12 is tested from l >= 1)
    double tol;
    int rule;
    int slot;
    int *executed;                      // ctrl[0] <- slot + 1 by every iteration that runs
};

struct IterParams {
    StopCheck stop;
    int J, N, G, n;
    int bc_left, bc_right;
    const double *Minv;
    const double *c;
    const double *psi_old;
    double *psi_new;
    double *phi;
    const double *mu, *w;
    const double *inc_left, *inc_right;
    unsigned long long *resid_inf; // slot of this iteration
    double *resid_l2;              // slot of this iteration (nullptr: not recorded)
    // work decomposition of the pipelined kernel
    int cpb;      // cells per work item (> 1 only when a whole item fits one chunk)
    int S;        // column sub-groups per cell team
    int cw;       // columns per chunk (cpb == 1)
    int nch;      // chunks per item
    int n_items;
    int stages;   // matrix ring depth
    int chunk_doubles;
    int color, ncolors;   // structured path: cells j = ncolors * i + color (ncolors = 1: all cells)
    int reverse;  // warp-per-cell kernel: every CTA walks its range of cells from the top down (see iterate.cu)
};

// opt-in dynamic shared memory for `fn`, once per (context, kernel, size)
static inline cudaError_t grant_smem(oci_ctx *ctx, int slot, const void *fn, size_t smem)
{
    if (ctx->smem_granted[slot] >= smem) return cudaSuccess;
    const cudaError_t e = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e == cudaSuccess) ctx->smem_granted[slot] = smem;
    return e;
}

// Every entry point of the C ABI works on the device the context was created on, whatever device is current in the
// calling thread; the caller's current device is restored on return.
struct DeviceGuard {
    int prev;
    bool switched;
    explicit DeviceGuard(int dev) : prev(dev), switched(false)
    {
        if (cudaGetDevice(&prev) == cudaSuccess && prev != dev) switched = cudaSetDevice(dev) == cudaSuccess;
    }
    ~DeviceGuard()
    {
        if (switched) cudaSetDevice(prev);
    }
};

static inline ProblemView make_view(const oci_ctx *c)
{
    ProblemView p;
    p.J = c->J; p.N = c->N; p.G = c->G; p.n = c->n; p.dt = c->dt;
    p.bc_left = c->bc_left; p.bc_right = c->bc_right;
    p.dx = c->dx; p.sigma_t = c->sigma_t; p.transfer = c->transfer; p.v = c->v; p.mu = c->mu; p.w = c->w;
    return p;
}

// launchers implemented in the kernel translation units (each returns the number of kernels launched, < 0 on error)
int launch_factor(oci_ctx *ctx);
int launch_assemble_one(oci_ctx *ctx, int cell, double *A_dev_rowmajor);
int launch_factor_input(oci_ctx *ctx, int cell, double *A_dev_rowmajor);
int launch_const_rhs(oci_ctx *ctx);
int launch_empty(oci_ctx *ctx);
int launch_oci_iteration(oci_ctx *ctx, int hist_slot, bool want_l2, bool check_prev);
StopCheck make_stop(const oci_ctx *ctx, int slot, bool check_prev);
int launch_advance(oci_ctx *ctx);
int launch_seed_iterate(oci_ctx *ctx);
int launch_scalar_flux(oci_ctx *ctx, const double *psi, double *phi);
int launch_si_setup(oci_ctx *ctx);
bool st_supported(const oci_ctx *ctx);
int launch_st_factor(oci_ctx *ctx);
int launch_st_iteration(oci_ctx *ctx, const struct IterParams &P, bool want_l2);
// `k` structured iterations (history slots slot0 .. slot0 + k - 1) in ONE cooperative launch; 0 = not applicable
int launch_st_multi(oci_ctx *ctx, int slot0, int k, bool want_l2, bool check_between);
int launch_dense_multi(oci_ctx *ctx, int slot0, int k, bool want_l2, bool check_between);
int launch_si_iteration(oci_ctx *ctx, int hist_slot, bool want_l2, bool check_prev);

#ifdef __CUDACC__
// Launch with programmatic stream serialisation: the kernel may be scheduled while its predecessor on the stream is
// still draining, which hides the launch latency and the tail of the predecessor behind this kernel's prologue
// (see pdl_wait below).
template <class... KArgs, class... Args>
static inline cudaError_t launch_pdl(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t stream, Args... args)
{
    cudaLaunchConfig_t cfg;
    memset(&cfg, 0, sizeof(cfg));
    cfg.gridDim = grid;
    cfg.blockDim = block;
    cfg.dynamicSmemBytes = smem;
    cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kernel, KArgs(args)...);
}

// ------------------------------------------------------------------------------------------------------------
// Device helpers
// ------------------------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

// non-negative doubles order like their bit patterns; NaN is mapped to +inf so it is never lost
__device__ __forceinline__ unsigned long long resid_bits(double d)
{
    if (!(d == d)) d = __longlong_as_double(0x7ff0000000000000LL);
    return (unsigned long long)__double_as_longlong(d);
}

// Same arithmetic, operation by operation, as the host test in step_impl (api.cu). COHERENT: the residual slots
// were written by other CTAs of the SAME launch (multi-iteration cooperative kernel), so read them past the L1.
template <bool COHERENT>
__device__ __forceinline__ bool stop_reached_t(const StopCheck &s)
{
    if (!s.prev_inf) return false;
    if (s.rule == OCI_STOP_DPHI_INF) {
        const unsigned long long b = COHERENT ? __ldcg(s.prev_inf) : *s.prev_inf;
        return __longlong_as_double((long long)b) < s.tol;
    }
    if (!s.prev2_l2) return false;
    const double e2 = COHERENT ? __ldcg(s.prev_l2) : *s.prev_l2, e2p = COHERENT ? __ldcg(s.prev2_l2) : *s.prev2_l2;
    if (e2 == 0.0 && e2p == 0.0) return true; // two skipped slots in a row
    const double e = __dsqrt_rn(e2), ep = __dsqrt_rn(e2p);
    return e < __dmul_rn(s.tol, __dsub_rn(1.0, __ddiv_rn(e, ep)));
}
__device__ __forceinline__ bool stop_reached(const StopCheck &s) { return stop_reached_t<false>(s); }

__device__ __forceinline__ double warp_max(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        double u = __shfl_xor_sync(0xffffffffu, v, o);
        v = (u > v || !(u == u)) ? u : v;
    }
    return v;
}

__device__ __forceinline__ double warp_sum(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// ---- programmatic dependent launch (the per-iteration kernels of one step follow each other on one stream) ----
// pdl_launch_dependents(): the next kernel of the stream may start launching (its CTAs take the SMs as ours leave);
// pdl_wait(): block until the previous kernel has completed and its writes are visible. A kernel launched with
// launch_pdl() must call pdl_wait() before it reads or writes anything the previous kernel touches. Both are no-ops in
// a kernel launched the ordinary way.
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

// ---- mbarrier / bulk-copy PTX wrappers ---------------------------------------------------------------------
__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void fence_mbar_init()
{
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t *bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t *bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint64_t *bar, uint32_t parity)
{
    uint32_t ok;
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
        "selp.u32 %0, 1, 0, p;\n"
        "}\n"
        : "=r"(ok)
        : "r"(smem_u32(bar)), "r"(parity)
        : "memory");
    return ok != 0;
}
// Bounded wait: a protocol bug traps (-> CUDA error) instead of hanging the GPU.
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity)
{
    if (mbar_try_wait(bar, parity)) return;
    unsigned long long t0 = 0;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t0));
    uint32_t spins = 0;
    while (!mbar_try_wait(bar, parity)) {
        if ((++spins & 0x3ff) == 0) {
            unsigned long long t1;
            asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t1));
            if (t1 - t0 > 4000000000ULL) __trap(); // 4 s
        }
    }
}
__device__ __forceinline__ void bulk_g2s(void *dst_smem, const void *src_gmem, uint32_t bytes, uint64_t *bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     smem_u32(dst_smem)),
                 "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}
// Eq. 8b, PAPER.md:132 -- entry (p, pp) of the 4x4 within-cell block L_{c,j,g,m}. Every operation is an
// explicitly rounded intrinsic so that the assembled matrix is bit-identical to a plain (uncontracted)
// evaluation of the same formula.
__device__ __forceinline__ double lc_entry(int p, int pp, double dx, double sig, double v, double dt, double mu)
{
    const double a = __dmul_rn(__dadd_rn(fabs(mu), __dmul_rn(dx, sig)), 0.5); // (|mu| + dx Sigma)/2
    const double gam = __ddiv_rn(dx, __dmul_rn(v, dt));                       // dx / (v dt)
    const double h = __dmul_rn(mu, 0.5);
    const int e = p * 4 + pp;
    switch (e) {
    case 0:  return a;
    case 1:  return h;
    case 2:  return __dmul_rn(gam, 0.5);
    case 4:  return -h;
    case 5:  return a;
    case 7:  return __dmul_rn(gam, 0.5);
    case 8:  return -gam;
    case 10: return __dadd_rn(gam, a);
    case 11: return h;
    case 13: return -gam;
    case 14: return -h;
    case 15: return __dadd_rn(gam, a);
    default: return 0.0;
    }
}
// ---- 4x4 inverse by Gauss-Jordan with partial pivoting, fully unrolled (registers only) ---------------------
// Returns false if a pivot was zero or not finite (the result is then meaningless).
__device__ __forceinline__ bool inv4(double (&a)[4][4], double (&b)[4][4])
{
    bool ok = true;
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
        ok = ok && fabs(a[k][k]) > 0.0 && fabs(a[k][k]) <= 1.7e308; // (NaN fails both)
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
    return ok;
}

#endif
