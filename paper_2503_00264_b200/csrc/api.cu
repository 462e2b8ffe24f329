// api.cu -- the C ABI of include/oci.h: workspace carving, state management, the convergence loops of
// Alg. 2 (OCI) and Alg. 1 (SI). Host logic only; every numerical step is a
// kernel in factor.cu / iterate.cu / si.cu.
#include "common.cuh"
#include <nvtx3/nvToolsExt.h> // header-only; ranges show up under nsys / ncu --nvtx, and cost nothing otherwise
#include <math.h>
#include <initializer_list>
#include <new>
#include <stdlib.h>
#include <string.h>
#include <vector>

size_t factor_scratch_bytes(int n, int num_sms, int max_smem_optin);

namespace {

struct NvtxRange { // RAII range on the calling thread (tracing)
    explicit NvtxRange(const char *name) { nvtxRangePushA(name); }
    ~NvtxRange() { nvtxRangePop(); }
};

thread_local int g_create_cuda_error = 0; // cudaError_t of the most recent failed oci_create of this thread

constexpr size_t ALIGN = 256;
inline size_t up(size_t b) { return (b + ALIGN - 1) & ~(ALIGN - 1); }

struct Carver {
    unsigned char *base;
    size_t off;
    template <typename T> T *take(size_t count)
    {
        T *p = base ? reinterpret_cast<T *>(base + off) : nullptr;
        off += up(count * sizeof(T));
        return p;
    }
};

void device_limits(int *num_sms, int *max_smem, int dev = -1)
{
    *num_sms = 148;        // B200
    *max_smem = 232448;    // 227 KB opt-in shared memory per CTA on sm_100
    if (dev >= 0 || cudaGetDevice(&dev) == cudaSuccess) {
        int v = 0;
        if (cudaDeviceGetAttribute(&v, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess && v > 0) *num_sms = v;
        if (cudaDeviceGetAttribute(&v, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev) == cudaSuccess && v > 0) *max_smem = v;
    } else {
        (void)cudaGetLastError();
    }
}

int validate(const oci_problem *p)
{
    if (!p) return -1;
    if (p->J < 1 || p->G < 1 || p->N < 2 || (p->N & 1)) return OCI_E_UNSUPPORTED;
    const long long n = 4LL * p->N * p->G;
    if (n > OCI_MAX_N) return OCI_E_UNSUPPORTED;
    if (!p->dx || !p->sigma_t || !p->transfer || !p->v || !p->mu || !p->w) return -1;
    if (!(p->dt > 0.0)) return -1;
    if (p->bc_left < 0 || p->bc_left > 2 || p->bc_right < 0 || p->bc_right > 2) return -1;
    for (int m = 0; m < p->N; ++m)
        if (!(p->mu[m] != 0.0)) return -1;
    if (p->bc_left == OCI_BC_REFLECTIVE || p->bc_right == OCI_BC_REFLECTIVE)
        for (int m = 0; m < p->N; ++m)
            if (p->mu[m] != -p->mu[p->N - 1 - m]) return -1;
    return 0;
}

// lays out the workspace; with base == nullptr only measures it
size_t carve(oci_ctx *c, unsigned char *base, int J, int N, int G, int num_sms, int max_smem)
{
    const size_t n = 4 * (size_t)N * G, GN = (size_t)G * N;
    Carver cv{base, 0};
    oci_ctx dummy;
    oci_ctx *t = c ? c : &dummy;
    t->dx = cv.take<double>(J);
    t->sigma_t = cv.take<double>((size_t)J * G);
    t->transfer = cv.take<double>((size_t)J * G * G);
    t->v = cv.take<double>(G);
    t->mu = cv.take<double>(N);
    t->w = cv.take<double>(N);
    t->q = cv.take<double>((size_t)J * G * 4);
    t->inc_left = cv.take<double>(GN * 2);
    t->inc_right = cv.take<double>(GN * 2);
    t->psi_prev = cv.take<double>((size_t)J * GN * 2);
    t->psi[0] = cv.take<double>((size_t)J * n);
    t->psi[1] = cv.take<double>((size_t)J * n);
    t->phi = cv.take<double>((size_t)J * G * 4);
    t->c = cv.take<double>((size_t)J * n);
    t->Minv = cv.take<double>((size_t)J * n * n);
    t->scratch_bytes = factor_scratch_bytes((int)n, num_sms, max_smem);
    t->scratch = cv.take<double>(t->scratch_bytes / sizeof(double));
    t->info = cv.take<int>(4);
    t->si_Linv = cv.take<double>((size_t)J * GN * 16);
    t->si_T = cv.take<double>((size_t)J * GN * 8);
    t->si_base = cv.take<double>((size_t)J * GN * 4);
    t->si_in = cv.take<double>((size_t)J * GN * 2);
    const size_t GNpad = (GN + 15) / 16 * 16; // room for any "si_lanes" grouping (4, 8, 16)
    t->si_T2sw = cv.take<double>((size_t)J * GNpad * 4);
    t->si_bsw = cv.take<double>((size_t)J * GNpad * 2);
    // scan mode: 6 doubles per thread prefix (one thread per 4 sweep steps) + per 1024-step block aggregate, per chain
    t->si_scan_bytes = (((size_t)J + 1023) / 1024) * GN * 257 * 6 * sizeof(double);
    t->si_scan = cv.take<double>(t->si_scan_bytes / sizeof(double));
    t->st_LinvT = cv.take<double>((size_t)J * GN * 8); // two of the four rows of every block inverse (structured.cu ST_LK)
    t->st_Wg = cv.take<double>((size_t)J * G * 16);
    t->st_Cinv = cv.take<double>((size_t)J * 16 * G * G);
    t->resid_inf = cv.take<unsigned long long>(OCI_RESID_CAP);
    t->resid_l2 = cv.take<double>(OCI_RESID_CAP);
    t->ctrl = cv.take<int>(4);
    return cv.off;
}

int reset_history(oci_ctx *ctx)
{
    OCI_CUDA_TRY(ctx, cudaMemsetAsync(ctx->ctrl, 0, sizeof(int) * 4, ctx->stream));
    // only the slots that iterations were issued for since the last reset (a step of 20 iterations clears 2 x 160 bytes,
    // not 2 x 512 KB); every other slot still holds the zero it was given at create or at an earlier reset
    const size_t dirty = (size_t)(ctx->hist_dirty < OCI_RESID_CAP ? ctx->hist_dirty : OCI_RESID_CAP);
    if (dirty) {
        OCI_CUDA_TRY(ctx, cudaMemsetAsync(ctx->resid_inf, 0, sizeof(unsigned long long) * dirty, ctx->stream));
        OCI_CUDA_TRY(ctx, cudaMemsetAsync(ctx->resid_l2, 0, sizeof(double) * dirty, ctx->stream));
    }
    ctx->hist_dirty = 0;
    ctx->hist_len = 0;
    ctx->hist_has_l2 = 0;
    return 0;
}

int ensure_const_rhs(oci_ctx *ctx, long long *launches)
{
    if (!ctx->c_valid) {
        int r = launch_const_rhs(ctx);
        if (r < 0) return r;
        *launches += r;
        ctx->c_valid = true;
    }
    return 0;
}

int ensure_si(oci_ctx *ctx, long long *launches)
{
    if (!ctx->si_valid) {
        int r = launch_si_setup(ctx);
        if (r < 0) return r;
        *launches += r;
        ctx->si_valid = true;
    }
    return 0;
}

// scheme 0 = OCI, 1 = SI
int one_iteration(oci_ctx *ctx, int scheme, int slot, bool want_l2, bool check_prev)
{
    return scheme == 0 ? launch_oci_iteration(ctx, slot, want_l2, check_prev)
                       : launch_si_iteration(ctx, slot, want_l2, check_prev);
}

// Iterations slot0 .. slot0 + k - 1 of one scheme; check_between: every iteration but the first looks at the residual of
// the one before it and skips itself once the stop rule held (device-side stop). Returns kernels launched.
int issue_batch(oci_ctx *ctx, int scheme, int slot0, int k, bool want_l2, bool check_between)
{
    if (slot0 + k > ctx->hist_dirty) ctx->hist_dirty = slot0 + k;
    if (scheme == 0) { // one cooperative launch for the whole batch, where that applies
        int r = launch_st_multi(ctx, slot0, k, want_l2, check_between);
        if (r != 0) return r;
        r = launch_dense_multi(ctx, slot0, k, want_l2, check_between);
        if (r != 0) return r;
    }
    int launches = 0;
    for (int i = 0; i < k; ++i) {
        const int r = one_iteration(ctx, scheme, slot0 + i, want_l2, check_between && i > 0);
        if (r < 0) return r;
        launches += r;
    }
    return launches;
}

// The stop rule on the host: slot l of the history h (rule 0: max|dphi|; rule 1: sums of squares). Same arithmetic,
// operation by operation, as stop_reached() on the device.
bool rule_holds(int rule, double tol, const double *h_inf, const double *h_l2, int l)
{
    if (rule == OCI_STOP_DPHI_INF) return h_inf[l] < tol;
    if (l < 1) return false;
    const double e = sqrt(h_l2[l]), ep = sqrt(h_l2[l - 1]);
    return e < tol * (1.0 - e / ep);
}

// a1 + a2 enqueued without a host round-trip: the kernels, their event pair and the copy of the singular-cell flag into
// pinned memory. factor_finish() reads the flag and the time once the stream has been synchronised (by oci_factor at
// once, by a step together with its first batch of iterations: one synchronisation instead of two).
int *factor_info_host(oci_ctx *ctx) { return reinterpret_cast<int *>(ctx->h_resid + 2 * OCI_RESID_CAP + 1); }

int factor_enqueue(oci_ctx *ctx)
{
    NvtxRange range(ctx->opt_solve_mode == 1 ? "oci_factor (structured)" : "oci_factor (dense)");
    OCI_CUDA_TRY(ctx, cudaEventRecord(ctx->evf0, ctx->stream));
    int r = ctx->opt_solve_mode == 1 ? launch_st_factor(ctx) : launch_factor(ctx);
    if (r < 0) return r;
    OCI_CUDA_TRY(ctx, cudaEventRecord(ctx->evf1, ctx->stream));
    OCI_CUDA_TRY(ctx, cudaMemcpyAsync(factor_info_host(ctx), ctx->info, sizeof(int), cudaMemcpyDeviceToHost, ctx->stream));
    ctx->last_launches[0] = r;
    return 0;
}

int factor_finish(oci_ctx *ctx)
{
    float ms = 0.f;
    OCI_CUDA_TRY(ctx, cudaEventElapsedTime(&ms, ctx->evf0, ctx->evf1));
    ctx->last_ms[0] = ms;
    const int info = *factor_info_host(ctx);
    ctx->factor_flagged = info != 0x7f7f7f7f;
    if (ctx->factor_flagged) return info; // 1-based index of the first singular cell
    ctx->factored = true;
    return 0;
}

int iterate_impl(oci_ctx *ctx, int scheme, int n_iters)
{
    if (!ctx) return -1;
    NvtxRange range(scheme == 0 ? "oci_iterate" : "si_iterate");
    if (n_iters < 0) return -2;
    long long launches = 0;
    int r;
    if (scheme == 0) {
        if (!ctx->factored) return OCI_E_STATE;
        if ((r = ensure_const_rhs(ctx, &launches)) < 0) return r;
    } else {
        if ((r = ensure_si(ctx, &launches)) < 0) return r;
    }
    if (ctx->hist_len + n_iters > OCI_RESID_CAP)
        if ((r = reset_history(ctx)) < 0) return r;
    if (n_iters > OCI_RESID_CAP) return -2;
    const int which = scheme == 0 ? 1 : 2;
    OCI_CUDA_TRY(ctx, cudaEventRecord(ctx->ev0, ctx->stream));
    r = issue_batch(ctx, scheme, ctx->hist_len, n_iters, false, false);
    if (r < 0) return r;
    launches += r;
    OCI_CUDA_TRY(ctx, cudaEventRecord(ctx->ev1, ctx->stream));
    ctx->hist_len += n_iters;
    ctx->last_ms[which] = -1.0; // resolved lazily by oci_last_timing
    ctx->last_launches[which] = launches;
    return 0;
}

int step_impl(oci_ctx *ctx, int scheme, double tol, int max_iters, int check_every, int rule, int advance,
              int32_t *iters_out, double *resid_out)
{
    if (!ctx) return -1;
    if (!(tol >= 0.0)) return -2;
    if (max_iters < 1 || max_iters > OCI_RESID_CAP) return -3;
    if (check_every < 1) return -4;
    if (rule != OCI_STOP_DPHI_INF && rule != OCI_STOP_PAPER) return -5;
    NvtxRange range(scheme == 0 ? "oci_step" : "si_step");
    long long launches = 0;
    int r;
    if (ctx->opt_refactor_every_step) { // Alg. 2 as printed: `_gesv` in the first iteration of every step
        if (scheme == 0) ctx->factored = false;
        else ctx->si_valid = false;
    }
    bool factor_pending = false;
    if (scheme == 0) {
        if (!ctx->factored) { // enqueued here, checked with the first batch's read-back below
            if ((r = factor_enqueue(ctx)) < 0) return r;
            launches += ctx->last_launches[0];
            factor_pending = true;
        }
        if ((r = ensure_const_rhs(ctx, &launches)) < 0) return r;
    } else {
        if ((r = ensure_si(ctx, &launches)) < 0) return r;
    }
    if ((r = reset_history(ctx)) < 0) return r;
    const bool want_l2 = rule == OCI_STOP_PAPER;
    ctx->hist_has_l2 = want_l2;
    const int which = scheme == 0 ? 1 : 2;
    int it = 0, conv_at = 0;
    double last = INFINITY, kernel_ms = 0.0;
    ctx->stop_tol = tol;
    ctx->stop_rule = rule;
    double *h_inf = ctx->h_resid, *h_l2 = ctx->h_resid + OCI_RESID_CAP;
    int *h_exec = reinterpret_cast<int *>(ctx->h_resid + 2 * OCI_RESID_CAP);
    while (it < max_iters && !conv_at) {
        const int k = (max_iters - it < check_every) ? max_iters - it : check_every;
        NvtxRange batch(scheme == 0 ? "oci iteration batch" : "si iteration batch");
        OCI_CUDA_TRY(ctx, cudaEventRecord(ctx->ev0, ctx->stream));
        // slot it + i > it looks at slot it + i - 1 on the device and skips itself once the rule held
        r = issue_batch(ctx, scheme, it, k, want_l2, true);
        if (r < 0) return r;
        launches += r;
        OCI_CUDA_TRY(ctx, cudaEventRecord(ctx->ev1, ctx->stream));
        // the one host round-trip: k residuals + the executed-iterations counter, once every k iterations
        OCI_CUDA_TRY(ctx, cudaMemcpyAsync(h_inf + it, ctx->resid_inf + it, sizeof(double) * k, cudaMemcpyDeviceToHost,
                                          ctx->stream));
        if (want_l2)
            OCI_CUDA_TRY(ctx, cudaMemcpyAsync(h_l2 + it, ctx->resid_l2 + it, sizeof(double) * k, cudaMemcpyDeviceToHost,
                                              ctx->stream));
        OCI_CUDA_TRY(ctx, cudaMemcpyAsync(h_exec, ctx->ctrl, sizeof(int), cudaMemcpyDeviceToHost, ctx->stream));
        OCI_CUDA_TRY(ctx, cudaStreamSynchronize(ctx->stream));
        if (factor_pending) {
            factor_pending = false;
            if ((r = factor_finish(ctx)) != 0) {
                // A singular cell: this batch's iterations ran on a zeroed block and both Jacobi buffers, phi and the
                // residual slots hold their results. Leave a DEFINED state behind instead: the iterate as oci_set_state
                // leaves it (both time levels = psi_{k-1/2}, which was not touched), its phi, an empty history. A caller
                // that catches the code and retries with another dt starts from there.
                int r2 = launch_seed_iterate(ctx);
                if (r2 < 0) return r2;
                if ((r2 = launch_scalar_flux(ctx, ctx->psi[ctx->cur], ctx->phi)) < 0) return r2;
                if ((r2 = reset_history(ctx)) < 0) return r2;
                ctx->last_ms[which] = 0.0;
                ctx->last_launches[which] = launches + 2;
                if (iters_out) { iters_out[0] = 0; iters_out[1] = 0; }
                if (resid_out) *resid_out = INFINITY;
                return r;
            }
        }
        {
            float t = 0.f; // device time of this batch of k launches (kernels only, no flag read)
            OCI_CUDA_TRY(ctx, cudaEventElapsedTime(&t, ctx->ev0, ctx->ev1));
            kernel_ms += t;
        }
        const int executed = *h_exec; // iterations of this step that really ran (<= it + k)
        if (executed < it + 1 || executed > it + k) return OCI_E_STATE;
        // skipped launches did not swap the Jacobi buffers (red-black works in place: nothing to undo)
        if (scheme == 0 && ctx->opt_ordering == 0 && ((it + k - executed) & 1)) ctx->cur ^= 1;
        const int l = executed - 1;
        last = want_l2 ? sqrt(h_l2[l]) : h_inf[l];
        if (executed < it + k) conv_at = executed;                       // the device saw the rule hold at slot l
        else if (rule_holds(rule, tol, h_inf, h_l2, l)) conv_at = executed; // last slot of the batch: tested here
        it = executed;
    }
    ctx->hist_len = it;
    ctx->last_ms[which] = kernel_ms;
    ctx->last_launches[which] = launches;
    if (advance) {
        r = launch_advance(ctx);
        if (r < 0) return r;
        ctx->last_launches[which] += r;
        ctx->c_valid = false;
    }
    // (no synchronisation here: the advance kernel is stream-ordered before anything the caller enqueues next)
    if (iters_out) { iters_out[0] = it; iters_out[1] = conv_at; }
    if (resid_out) *resid_out = last;
    return 0;
}

} // namespace

StopCheck make_stop(const oci_ctx *ctx, int slot, bool check_prev)
{
    StopCheck s;
    const bool chk = check_prev && slot >= 1;
    s.prev_inf = chk ? ctx->resid_inf + slot - 1 : nullptr;
    s.prev_l2 = chk ? ctx->resid_l2 + slot - 1 : nullptr;
    s.prev2_l2 = (chk && slot >= 2) ? ctx->resid_l2 + slot - 2 : nullptr;
    s.tol = ctx->stop_tol;
    s.rule = ctx->stop_rule;
    s.slot = slot;
    s.executed = ctx->ctrl;
    return s;
}

extern "C" {

size_t oci_workspace_bytes(const oci_problem *p)
{
    if (validate(p) != 0) return 0;
    int sms, smem;
    device_limits(&sms, &smem);
    return carve(nullptr, nullptr, p->J, p->N, p->G, sms, smem);
}

int oci_create(const oci_problem *p, void *workspace_dev, size_t workspace_bytes, void *cuda_stream, oci_ctx **out)
{
    if (!out) return -5;
    *out = nullptr;
    int v = validate(p);
    if (v != 0) return v;
    if (!workspace_dev) return -2;
    if (((uintptr_t)workspace_dev) % ALIGN) return OCI_E_WORKSPACE;
    oci_ctx *ctx = new (std::nothrow) oci_ctx();
    if (!ctx) return OCI_E_NOMEM;
    memset(ctx, 0, sizeof(*ctx));
    ctx->J = p->J; ctx->N = p->N; ctx->G = p->G; ctx->n = 4 * p->N * p->G;
    ctx->dt = p->dt; ctx->bc_left = p->bc_left; ctx->bc_right = p->bc_right;
    ctx->stream = (cudaStream_t)cuda_stream;
    ctx->opt_iterate_kernel = 1;
    ctx->opt_factor_kernel = 1;
    ctx->opt_factor_update = 2;
    ctx->opt_persistent = -1;
    ctx->opt_st_warp_local = 1;
    ctx->opt_st_fused_setup = 1;
    g_create_cuda_error = 0;
    auto fail = [&](int code) { // keeps the CUDA error retrievable: oci_last_create_error()
        if (code == OCI_E_CUDA) {
            g_create_cuda_error = (int)cudaGetLastError();
            if (g_create_cuda_error == 0) g_create_cuda_error = ctx->last_cuda ? ctx->last_cuda : (int)cudaErrorUnknown;
        }
        oci_destroy(ctx);
        return code;
    };
    // the context lives on the device that owns the workspace, whatever device is current in the calling thread
    {
        cudaPointerAttributes pa;
        if (cudaPointerGetAttributes(&pa, workspace_dev) != cudaSuccess) return fail(OCI_E_CUDA);
        if (pa.type != cudaMemoryTypeDevice && pa.type != cudaMemoryTypeManaged) { oci_destroy(ctx); return -2; }
        ctx->device = pa.device;
    }
    DeviceGuard guard(ctx->device);
    device_limits(&ctx->num_sms, &ctx->max_smem_optin, ctx->device);
    const size_t need = carve(ctx, (unsigned char *)workspace_dev, p->J, p->N, p->G, ctx->num_sms, ctx->max_smem_optin);
    if (need > workspace_bytes) return fail(OCI_E_WORKSPACE);
    if (cudaHostAlloc((void **)&ctx->h_resid, sizeof(double) * (2 * OCI_RESID_CAP + 4), cudaHostAllocDefault) != cudaSuccess)
        return fail(OCI_E_CUDA);
    if (cudaEventCreate(&ctx->ev0) != cudaSuccess || cudaEventCreate(&ctx->ev1) != cudaSuccess) return fail(OCI_E_CUDA);
    if (cudaEventCreate(&ctx->evf0) != cudaSuccess || cudaEventCreate(&ctx->evf1) != cudaSuccess) return fail(OCI_E_CUDA);
    cudaStream_t s = ctx->stream;
    const size_t J = p->J, G = p->G, N = p->N, n = ctx->n;
#define UP(dst, src, cnt)                                                                                      \
    if (cudaMemcpyAsync(dst, src, sizeof(double) * (cnt), cudaMemcpyHostToDevice, s) != cudaSuccess) return fail(OCI_E_CUDA)
    UP(ctx->dx, p->dx, J);
    UP(ctx->sigma_t, p->sigma_t, J * G);
    UP(ctx->transfer, p->transfer, J * G * G);
    UP(ctx->v, p->v, G);
    UP(ctx->mu, p->mu, N);
    UP(ctx->w, p->w, N);
#undef UP
#define ZERO(dst, bytes) \
    if (cudaMemsetAsync(dst, 0, bytes, s) != cudaSuccess) return fail(OCI_E_CUDA)
    ZERO(ctx->q, sizeof(double) * J * G * 4);
    ZERO(ctx->inc_left, sizeof(double) * G * N * 2);
    ZERO(ctx->inc_right, sizeof(double) * G * N * 2);
    ZERO(ctx->psi_prev, sizeof(double) * J * G * N * 2);
    ZERO(ctx->psi[0], sizeof(double) * J * n);
    ZERO(ctx->psi[1], sizeof(double) * J * n);
    ZERO(ctx->phi, sizeof(double) * J * G * 4);
    ZERO(ctx->resid_inf, sizeof(double) * OCI_RESID_CAP);
    ZERO(ctx->resid_l2, sizeof(double) * OCI_RESID_CAP);
    ZERO(ctx->ctrl, sizeof(int) * 4);
#undef ZERO
    if (cudaStreamSynchronize(s) != cudaSuccess) return fail(OCI_E_CUDA);
    *out = ctx;
    return 0;
}

void oci_destroy(oci_ctx *ctx)
{
    if (!ctx) return;
    DeviceGuard guard(ctx->device);
    if (ctx->h_resid) cudaFreeHost(ctx->h_resid);
    if (ctx->ev0) cudaEventDestroy(ctx->ev0);
    if (ctx->ev1) cudaEventDestroy(ctx->ev1);
    if (ctx->evf0) cudaEventDestroy(ctx->evf0);
    if (ctx->evf1) cudaEventDestroy(ctx->evf1);
    delete ctx;
}

const char *oci_strerror(int code)
{
    switch (code) {
    case 0: return "ok";
    case OCI_E_CUDA: return "CUDA call or kernel failed";
    case OCI_E_WORKSPACE: return "workspace too small or misaligned";
    case OCI_E_UNSUPPORTED: return "problem outside the supported range";
    case OCI_E_STATE: return "call order violated";
    case OCI_E_NOMEM: return "host allocation failed";
    case OCI_E_TOO_LARGE: return "J * G exceeds OCI_STATIC_MAX_PAIRS: the no-allocation entry point has a fixed scratch array";
    default: return code > 0 ? "singular cell matrix (value = 1-based cell index)" : "invalid argument (value = -index)";
    }
}

int oci_last_cuda_error(const oci_ctx *ctx) { return ctx ? ctx->last_cuda : 0; }
int oci_last_create_error(void) { return g_create_cuda_error; }

int oci_set_option(oci_ctx *ctx, const char *key, int64_t value)
{
    if (!ctx) return -1;
    DeviceGuard guard(ctx->device);
    if (!key) return -2;
    // stale factors also means a stale "some cells were singular" record: oci_debug_get_inverse must not serve the
    // inverses of another dt / another kernel after it
    auto drop_factors = [&]() { ctx->factored = false; ctx->factor_flagged = false; };
    auto in = [&](std::initializer_list<int64_t> ok) {
        for (int64_t v : ok)
            if (v == value) return true;
        return false;
    };
    if (!strcmp(key, "iterate_kernel")) {
        if (!in({0, 1})) return -3;
        ctx->opt_iterate_kernel = (int)value;
    }
    else if (!strcmp(key, "iterate_stages")) {
        if (value < 0 || value > 64) return -3; // 0 = as many as fit
        ctx->opt_stages = (int)value;
    }
    else if (!strcmp(key, "factor_kernel")) {
        if (!in({0, 1, 4})) return -3;
        ctx->opt_factor_kernel = (int)value;
        drop_factors();
    }
    else if (!strcmp(key, "factor_update")) {
        if (!in({0, 1, 2})) return -3;
        ctx->opt_factor_update = (int)value;
        drop_factors();
    }
    else if (!strcmp(key, "factor_cluster")) {
        if (!in({0, 1})) return -3;
        ctx->opt_factor_cluster = (int)value;
        drop_factors();
    }
    else if (!strcmp(key, "refactor_every_step")) {
        if (!in({0, 1})) return -3;
        ctx->opt_refactor_every_step = (int)value;
    }
    else if (!strcmp(key, "solve_mode")) {
        if (value != 0 && value != 1) return -3;
        if (value == 1 && !st_supported(ctx)) return OCI_E_UNSUPPORTED;
        if ((int)value != ctx->opt_solve_mode) drop_factors();
        ctx->opt_solve_mode = (int)value;
    }
    else if (!strcmp(key, "ordering")) {
        if (value != 0 && value != 1) return -3;
        ctx->opt_ordering = (int)value;
    }
    else if (!strcmp(key, "persistent")) { // -1 auto, 0 off, 1 on (structured path)
        if (!in({-1, 0, 1})) return -3;
        ctx->opt_persistent = (int)value;
    }
    else if (!strcmp(key, "si_sweep")) {
        if (value != 0 && value != 1) return -3;
        if ((int)value != ctx->opt_si_sweep) ctx->si_valid = false; // the sweep-order arrays change layout
        ctx->opt_si_sweep = (int)value;
    }
    else if (!strcmp(key, "si_lanes")) {
        if (!in({0, 4, 8, 16})) return -3; // 0 = default (8)
        ctx->opt_si_lanes = (int)value;
        ctx->si_valid = false;
    }
    else return -2;
    return 0;
}

int oci_set_dt(oci_ctx *ctx, double dt)
{
    if (!ctx) return -1;
    DeviceGuard guard(ctx->device);
    if (!(dt > 0.0)) return -2;
    if (dt != ctx->dt) {
        ctx->dt = dt;
        ctx->factored = false;
        ctx->factor_flagged = false;
        ctx->si_valid = false;
        ctx->c_valid = false;
    }
    return 0;
}

int oci_set_source(oci_ctx *ctx, const double *q_dev)
{
    if (!ctx) return -1;
    DeviceGuard guard(ctx->device);
    const size_t bytes = sizeof(double) * (size_t)ctx->J * ctx->G * 4;
    if (q_dev) OCI_CUDA_TRY(ctx, cudaMemcpyAsync(ctx->q, q_dev, bytes, cudaMemcpyDeviceToDevice, ctx->stream));
    else OCI_CUDA_TRY(ctx, cudaMemsetAsync(ctx->q, 0, bytes, ctx->stream));
    ctx->c_valid = false;
    return 0;
}

int oci_set_incident(oci_ctx *ctx, const double *left_dev, const double *right_dev)
{
    if (!ctx) return -1;
    DeviceGuard guard(ctx->device);
    const size_t bytes = sizeof(double) * (size_t)ctx->G * ctx->N * 2;
    if (left_dev) OCI_CUDA_TRY(ctx, cudaMemcpyAsync(ctx->inc_left, left_dev, bytes, cudaMemcpyDeviceToDevice, ctx->stream));
    if (right_dev) OCI_CUDA_TRY(ctx, cudaMemcpyAsync(ctx->inc_right, right_dev, bytes, cudaMemcpyDeviceToDevice, ctx->stream));
    return 0;
}

int oci_set_state(oci_ctx *ctx, const double *psi_edge_dev)
{
    if (!ctx) return -1;
    DeviceGuard guard(ctx->device);
    if (!psi_edge_dev) return -2;
    const size_t bytes = sizeof(double) * (size_t)ctx->J * ctx->G * ctx->N * 2;
    OCI_CUDA_TRY(ctx, cudaMemcpyAsync(ctx->psi_prev, psi_edge_dev, bytes, cudaMemcpyDeviceToDevice, ctx->stream));
    int r = launch_seed_iterate(ctx);
    if (r < 0) return r;
    r = launch_scalar_flux(ctx, ctx->psi[ctx->cur], ctx->phi);
    if (r < 0) return r;
    ctx->c_valid = false;
    return 0;
}

int oci_get_state(oci_ctx *ctx, double *psi_edge_dev)
{
    if (!ctx) return -1;
    DeviceGuard guard(ctx->device);
    if (!psi_edge_dev) return -2;
    const size_t bytes = sizeof(double) * (size_t)ctx->J * ctx->G * ctx->N * 2;
    OCI_CUDA_TRY(ctx, cudaMemcpyAsync(psi_edge_dev, ctx->psi_prev, bytes, cudaMemcpyDeviceToDevice, ctx->stream));
    return 0;
}

int oci_set_iterate(oci_ctx *ctx, const double *psi_dev)
{
    if (!ctx) return -1;
    DeviceGuard guard(ctx->device);
    if (!psi_dev) return -2;
    const size_t bytes = sizeof(double) * (size_t)ctx->J * ctx->n;
    OCI_CUDA_TRY(ctx, cudaMemcpyAsync(ctx->psi[ctx->cur], psi_dev, bytes, cudaMemcpyDeviceToDevice, ctx->stream));
    int r = launch_scalar_flux(ctx, ctx->psi[ctx->cur], ctx->phi);
    return r < 0 ? r : 0;
}

int oci_factor(oci_ctx *ctx)
{
    if (!ctx) return -1;
    DeviceGuard guard(ctx->device);
    if (ctx->factored) return 0;
    int r = factor_enqueue(ctx);
    if (r < 0) return r;
    OCI_CUDA_TRY(ctx, cudaStreamSynchronize(ctx->stream));
    return factor_finish(ctx);
}

int oci_iterate(oci_ctx *ctx, int32_t n_iters)
{
    if (!ctx) return -1;
    DeviceGuard guard(ctx->device);
    return iterate_impl(ctx, 0, n_iters);
}
int si_iterate(oci_ctx *ctx, int32_t n_iters)
{
    if (!ctx) return -1;
    DeviceGuard guard(ctx->device);
    return iterate_impl(ctx, 1, n_iters);
}

int oci_step(oci_ctx *ctx, double tol, int32_t max_iters, int32_t check_every, int32_t stop_rule, int32_t advance,
             int32_t *iters_out, double *resid_out)
{
    if (!ctx) return -1;
    DeviceGuard guard(ctx->device);
    return step_impl(ctx, 0, tol, max_iters, check_every, stop_rule, advance, iters_out, resid_out);
}

int si_step(oci_ctx *ctx, double tol, int32_t max_iters, int32_t check_every, int32_t stop_rule, int32_t advance,
            int32_t *iters_out, double *resid_out)
{
    if (!ctx) return -1;
    DeviceGuard guard(ctx->device);
    return step_impl(ctx, 1, tol, max_iters, check_every, stop_rule, advance, iters_out, resid_out);
}

int oci_advance(oci_ctx *ctx)
{
    if (!ctx) return -1;
    DeviceGuard guard(ctx->device);
    int r = launch_advance(ctx);
    if (r < 0) return r;
    ctx->c_valid = false;
    return 0;
}

int oci_scalar_flux(oci_ctx *ctx, double *phi_dev)
{
    if (!ctx) return -1;
    DeviceGuard guard(ctx->device);
    if (!phi_dev) return -2;
    OCI_CUDA_TRY(ctx, cudaMemcpyAsync(phi_dev, ctx->phi, sizeof(double) * (size_t)ctx->J * ctx->G * 4,
                                      cudaMemcpyDeviceToDevice, ctx->stream));
    return 0;
}

int oci_angular_flux(oci_ctx *ctx, double *psi_dev)
{
    if (!ctx) return -1;
    DeviceGuard guard(ctx->device);
    if (!psi_dev) return -2;
    OCI_CUDA_TRY(ctx, cudaMemcpyAsync(psi_dev, ctx->psi[ctx->cur], sizeof(double) * (size_t)ctx->J * ctx->n,
                                      cudaMemcpyDeviceToDevice, ctx->stream));
    return 0;
}

int oci_residual_history(oci_ctx *ctx, int32_t kind, double *host_out, int32_t cap, int32_t *n)
{
    if (!ctx) return -1;
    DeviceGuard guard(ctx->device);
    if (kind != 0 && kind != 1) return -2;
    if (!n) return -5;
    const int len = ctx->hist_len;
    *n = len;
    if (!host_out || cap <= 0 || len == 0) return 0;
    const int cnt = len < cap ? len : cap;
    const void *src = kind == 0 ? (const void *)ctx->resid_inf : (const void *)ctx->resid_l2;
    OCI_CUDA_TRY(ctx, cudaMemcpyAsync(host_out, src, sizeof(double) * cnt, cudaMemcpyDeviceToHost, ctx->stream));
    OCI_CUDA_TRY(ctx, cudaStreamSynchronize(ctx->stream));
    if (kind == 1)
        for (int i = 0; i < cnt; ++i) host_out[i] = sqrt(host_out[i]);
    return 0;
}

int oci_step_host(oci_ctx *ctx, int32_t scheme, const double *q_host, double tol, int32_t max_iters,
                  int32_t check_every, int32_t stop_rule, int32_t advance, int32_t *iters_out, double *resid_out,
                  double *phi_host)
{
    if (!ctx) return -1;
    DeviceGuard guard(ctx->device);
    if (scheme != 0 && scheme != 1) return -2;
    const size_t bytes = sizeof(double) * (size_t)ctx->J * ctx->G * 4;
    if (q_host) {
        OCI_CUDA_TRY(ctx, cudaMemcpyAsync(ctx->q, q_host, bytes, cudaMemcpyHostToDevice, ctx->stream));
        ctx->c_valid = false;
    }
    int r = step_impl(ctx, scheme, tol, max_iters, check_every, stop_rule, advance, iters_out, resid_out);
    if (r != 0) return r;
    if (phi_host) {
        OCI_CUDA_TRY(ctx, cudaMemcpyAsync(phi_host, ctx->phi, bytes, cudaMemcpyDeviceToHost, ctx->stream));
        OCI_CUDA_TRY(ctx, cudaStreamSynchronize(ctx->stream));
    }
    return 0;
}

int oci_debug_get_matrix(oci_ctx *ctx, int32_t cell, double *A_host)
{
    if (!ctx) return -1;
    DeviceGuard guard(ctx->device);
    if (cell < 0 || cell >= ctx->J) return -2;
    if (!A_host) return -3;
    int r = launch_assemble_one(ctx, cell, ctx->scratch);
    if (r < 0) return r;
    OCI_CUDA_TRY(ctx, cudaMemcpyAsync(A_host, ctx->scratch, sizeof(double) * (size_t)ctx->n * ctx->n,
                                      cudaMemcpyDeviceToHost, ctx->stream));
    OCI_CUDA_TRY(ctx, cudaStreamSynchronize(ctx->stream));
    return 0;
}

int oci_debug_get_factor_input(oci_ctx *ctx, int32_t cell, double *A_host)
{
    if (!ctx) return -1;
    DeviceGuard guard(ctx->device);
    if (cell < 0 || cell >= ctx->J) return -2;
    if (!A_host) return -3;
    int r = launch_factor_input(ctx, cell, ctx->scratch);
    if (r < 0) return r;
    if (r == 0) return OCI_E_UNSUPPORTED;
    OCI_CUDA_TRY(ctx, cudaMemcpyAsync(A_host, ctx->scratch, sizeof(double) * (size_t)ctx->n * ctx->n,
                                      cudaMemcpyDeviceToHost, ctx->stream));
    OCI_CUDA_TRY(ctx, cudaStreamSynchronize(ctx->stream));
    return 0;
}

int oci_debug_get_inverse(oci_ctx *ctx, int32_t cell, double *Ainv_host)
{
    if (!ctx) return -1;
    DeviceGuard guard(ctx->device);
    if (cell < 0 || cell >= ctx->J) return -2;
    if (!Ainv_host) return -3;
    if (!ctx->factored && !ctx->factor_flagged) return OCI_E_STATE;
    if (ctx->opt_solve_mode == 1) return OCI_E_UNSUPPORTED; // the structured path never forms A_j^{-1}
    const size_t n = ctx->n;
    std::vector<double> tmp(n * n);
    OCI_CUDA_TRY(ctx, cudaMemcpyAsync(tmp.data(), ctx->Minv + (size_t)cell * n * n, sizeof(double) * n * n,
                                      cudaMemcpyDeviceToHost, ctx->stream));
    OCI_CUDA_TRY(ctx, cudaStreamSynchronize(ctx->stream));
    for (size_t r = 0; r < n; ++r)
        for (size_t c = 0; c < n; ++c) Ainv_host[r * n + c] = tmp[c * n + r]; // stored column-major
    return 0;
}

int oci_debug_get_const_rhs(oci_ctx *ctx, double *c_dev)
{
    if (!ctx) return -1;
    DeviceGuard guard(ctx->device);
    if (!c_dev) return -2;
    long long l = 0;
    int r = ensure_const_rhs(ctx, &l);
    if (r < 0) return r;
    OCI_CUDA_TRY(ctx, cudaMemcpyAsync(c_dev, ctx->c, sizeof(double) * (size_t)ctx->J * ctx->n, cudaMemcpyDeviceToDevice,
                                      ctx->stream));
    return 0;
}

int oci_debug_empty_launches(oci_ctx *ctx, int32_t count)
{
    if (!ctx) return -1;
    DeviceGuard guard(ctx->device);
    if (count < 0) return -2;
    for (int i = 0; i < count; ++i) {
        int r = launch_empty(ctx);
        if (r < 0) return r;
    }
    return 0;
}

int oci_last_timing(oci_ctx *ctx, int32_t which, double *ms, int64_t *launches)
{
    if (!ctx) return -1;
    DeviceGuard guard(ctx->device);
    if (which < 0 || which > 2) return -2;
    if (ctx->last_ms[which] < 0.0) {
        // ev0/ev1 bracket the most recent iterate / step call; valid only if `which` was that call
        OCI_CUDA_TRY(ctx, cudaEventSynchronize(ctx->ev1));
        float t = 0.f;
        OCI_CUDA_TRY(ctx, cudaEventElapsedTime(&t, ctx->ev0, ctx->ev1));
        ctx->last_ms[which] = t;
    }
    if (ms) *ms = ctx->last_ms[which];
    if (launches) *launches = ctx->last_launches[which];
    return 0;
}

} // extern "C"
