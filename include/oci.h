/*
 * oci.h -- C ABI of the B200 (sm_100a) one-cell-inversion (OCI) transport library, liboci_b200.so.
 *
 * The library is the data-parallel hot path of arXiv 2503.00264 ("One-Cell Inversion for Solving Higher-Order
 * Time-Dependent Radiation Transport on GPUs"): time-dependent 1-D slab multigroup S_N transport, simple corner
 * balance in space (Eq. 3a-d), multiple balance in time (Eq. 2a-b), solved per
 * time step by the cell-wise block-Jacobi OCI iteration (Eq. 6-7; Alg. 2),
 * with a source-iteration (SI) sweep (Appendix A, Eq. 42-46; Alg. 1) as
 * the comparator. Everything is fp64. There is no CPU fallback: every entry point that computes runs CUDA
 * kernels on the device the workspace lives on, and fails with OCI_E_CUDA if it cannot.
 *
 * Conventions
 *  - Every function returns int: 0 = OK; < 0 = error (OCI_E_*; -1..-9 = "argument i is bad");
 *    oci_factor additionally returns > 0 = 1-based index of the first cell whose elimination met a zero /
 *    NaN pivot (LAPACK `info` convention).
 *  - No exceptions, no stdout/stderr. The library never allocates device memory: the caller owns one
 *    workspace of oci_workspace_bytes() bytes (256-byte aligned) and keeps it alive until oci_destroy.
 *  - "host" / "dev" after an argument says where the pointer must live. Problem-description arrays are host
 *    pointers and are copied at oci_create. Device arrays passed in are read during the call's stream work
 *    and may be reused after the stream has passed that point; they are never kept.
 *  - All work is enqueued on the stream given at create time. Calls marked [async] return without
 *    synchronising; calls marked [sync] synchronise that stream before returning.
 *
 * Layouts (Eq. 11a-b, 40c-d), all fp64, C-contiguous:
 *   n = 4*N*G unknowns per cell, index r = (g*N + m)*4 + p, p = 0:(k,L) 1:(k,R) 2:(k+1/2,L) 3:(k+1/2,R)
 *   psi       [J][G][N][4]   angular flux iterate (both time levels)
 *   psi_edge  [J][G][N][2]   time-edge angular flux psi_{k-1/2} at (L,R)
 *   phi       [J][G][4]      scalar flux phi = sum_m w_m psi_m (Eq. 44)
 *   q         [J][G][4]      isotropic source Q at (k,L) (k,R) (k+1/2,L) (k+1/2,R)
 *   incident  [G][N][2]      prescribed incident flux per ordinate at levels (k, k+1/2); only the ordinates
 *                            entering through that face are read (mu_m > 0 on the left, mu_m < 0 on the right)
 */
#ifndef OCI_B200_H
#define OCI_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define OCI_BC_VACUUM 0
#define OCI_BC_REFLECTIVE 1 /* mirror ordinate N-1-m, lagged one iteration (reading A12) */
#define OCI_BC_PRESCRIBED 2

#define OCI_E_ARG_BASE 0        /* -i : i-th argument invalid (1-based) */
#define OCI_E_CUDA (-100)       /* a CUDA call or kernel failed; oci_last_cuda_error() has the code */
#define OCI_E_WORKSPACE (-101)  /* workspace too small or misaligned */
#define OCI_E_UNSUPPORTED (-102)/* problem outside the supported range (N odd, n > OCI_MAX_N, ...) */
#define OCI_E_STATE (-103)      /* call order violated (e.g. iterate before factor) */
#define OCI_E_NOMEM (-104)      /* host allocation failed */
#define OCI_E_TOO_LARGE (-105)  /* oci_flux_residual_static: J * G beyond OCI_STATIC_MAX_PAIRS (its scratch is fixed) */

#define OCI_MAX_N 256           /* largest per-cell system order n = 4*N*G */
#define OCI_RESID_CAP 65536     /* residual history entries kept per time step */

#define OCI_STOP_DPHI_INF 0     /* max_{j,g,p} |phi^(l+1) - phi^(l)| < tol         (BASELINE.json configs) */
#define OCI_STOP_PAPER 1        /* Eq. 12-13: e_l < tol (1 - e_l / e_{l-1}), l >= 1      */

typedef struct oci_ctx oci_ctx;

/* Problem statement: Eq. 1 + IC/BC. All pointers are HOST pointers, copied at create. */
typedef struct {
    int32_t J, N, G;       /* cells, ordinates (even), groups */
    const double *dx;      /* [J] cell widths, cm */
    const double *sigma_t; /* [J][G] total cross-section, 1/cm */
    const double *transfer;/* [J][G_to][G_from] = Sigma_s(from->to) + chi_to nuSigma_f,from (Eq. 40b; reading A13) */
    const double *v;       /* [G] speeds, cm/s */
    const double *mu;      /* [N] quadrature nodes, no zero, mu[N-1-m] = -mu[m] if a face is reflective */
    const double *w;       /* [N] weights, sum = 2 (Eq. 1 normalisation, reading A8) */
    double dt;             /* time step, s */
    int32_t bc_left, bc_right;
} oci_problem;

/* Bytes of device workspace oci_create needs for this problem (0 if the problem is unsupported). */
size_t oci_workspace_bytes(const oci_problem *p);

/* Validates the problem, carves the workspace, uploads the problem arrays. State starts as psi = 0, q = 0.
 * cuda_stream is a cudaStream_t (NULL = legacy default stream) of the device the workspace lives on. The context is
 * bound to that device: every later call switches to it for its own duration and restores the caller's current
 * device, so contexts on several GPUs can be driven from one thread. [sync] */
int oci_create(const oci_problem *p, void *workspace_dev, size_t workspace_bytes, void *cuda_stream,
               oci_ctx **out);
void oci_destroy(oci_ctx *ctx);
const char *oci_strerror(int code);
int oci_last_cuda_error(const oci_ctx *ctx);
/* cudaError_t behind the most recent oci_create of the calling thread that returned OCI_E_CUDA (0 otherwise): a failed
 * create returns no context to ask. */
int oci_last_create_error(void);

/* Tuning knobs (all optional). Known keys: "iterate_kernel" (0 = plain one-CTA-per-cell, 1 = pipelined
 * bulk-copy streaming kernel [default]), "iterate_stages" (depth of its shared-memory ring, 0 [default] = as deep as
 * fits), "factor_kernel"
 * (0 = generic shared-memory elimination, one CTA per cell; 1 = production kernels [default]: for n = 64 the working
 * matrix in shared memory, one pivot warp + one update warp per cell with look-ahead and rank-8 updates on the FP64
 * tensor path (DMMA); for n = 128 the same with one CTA per cell (four pivot warps + four update warps); for n = 192,
 * 256 a thread-block cluster per cell, the working matrix in the cluster's distributed shared memory ("factor_cluster"
 * 0 [default] = as few CTAs as hold it, two at n = 192 and three at n = 256; 1 = n/64 CTAs of 64 columns each);
 * 4 = n = 64 with ONE warp per cell), "factor_update" (n = 64: 2 [default] = DMMA updates, a block that is
 * not needed soon receives the updates of two consecutive panels in one pass (rank 16); 1 = DMMA, one rank-8 pass per
 * panel; 0 = DFMA rank-8 updates, "factor_kernel" 4 only -- with 1 the A/B pair behind DESIGN.md's DMMA decision),
 * "solve_mode" (0 = dense
 * [default]: a2 eliminates the dense A_j with partial pivoting and a5 streams A_j^{-1}, the paper's method;
 * 1 = structured: A_j = D - U V^T with D the 4x4 blocks of Eq. 8b and rank 4G (Eq. 10 / 40b), a2 inverts the
 * blocks and the 4G x 4G capacitance matrix with partial pivoting, a5 applies them -- the same iteration to
 * rounding, 4n + 16 G^2 doubles of factors per cell-solve instead of n^2; needs G <= 8; switching invalidates the
 * factors), "refactor_every_step" (1 = oci_step / si_step redo
 * a1+a2 at the start of every step as Alg. 2 prints it; 0 [default] = only when dt changed), "si_lanes" (ordinates x
 * groups swept by one CTA of the SI sweep kernel: 4, 8 [default] or 16), "si_sweep" (0 = serial in space [default],
 * the comparator north_star names; 1 = the same sweep evaluated as a parallel scan of the per-cell affine edge maps,
 * same iterates to rounding), "persistent" (-1 [default] = run a batch of iterations as ONE
 * cooperative launch with grid-wide barriers when the problem is small: structured path <= 8 MB per iteration; dense
 * path when the inverses of ceil(J / SMs) cells fit in one CTA's shared memory, where they then stay for the whole
 * batch; 0 = never, 1 = always (structured path)), "ordering" (structured path only: 0 = block-Jacobi [default], the
 * paper's OCI; 1 = red-black: per iteration the even cells, then the odd cells from the new even ones, in place --
 * the block Gauss-Seidel variant PAPER.md:29, 550 names, about half the iterations; SURVEY.md 8(f) row f4;
 * oci_iterate / oci_step return OCI_E_UNSUPPORTED in the dense mode). Returns -2 for an unknown key, -3 for a bad
 * value. */
int oci_set_option(oci_ctx *ctx, const char *key, int64_t value);

int oci_set_dt(oci_ctx *ctx, double dt);                               /* invalidates the factors      */
int oci_set_source(oci_ctx *ctx, const double *q_dev);                 /* [J][G][4] dev; NULL = zero [async] */
int oci_set_incident(oci_ctx *ctx, const double *left_dev, const double *right_dev); /* [G][N][2] dev [async] */
/* psi_{k-1/2}; also seeds the iterate with both time levels = psi_edge (reading A11). [async] */
int oci_set_state(oci_ctx *ctx, const double *psi_edge_dev);
int oci_get_state(oci_ctx *ctx, double *psi_edge_dev);                 /* current psi_{k-1/2} [async]  */
/* Overrides the iterate Psi^(l) only (e.g. the random initial guess of PAPER.md:479). [async] */
int oci_set_iterate(oci_ctx *ctx, const double *psi_dev);

/* a1 + a2: assemble A_j = L_c - S (Eq. 8a-b, 10, 40b) for every cell
 * in on-chip memory and eliminate it with partial pivoting (what `_gesv` does in Alg. 2),
 * carried through to A_j^{-1}, which is what the iterate kernel streams. No-op if
 * the factors for the current dt are already present. [sync] (it reads back the singular-cell flag). */
int oci_factor(oci_ctx *ctx);

/* a3-a7: exactly n_iters block-Jacobi iterations (Eq. 7): b_j = c_j + incident(Psi^(l)),
 * Psi_j^(l+1) = A_j^{-1} b_j, phi^(l+1), residual. Builds the constant part c_j first if it is stale. [async] */
int oci_iterate(oci_ctx *ctx, int32_t n_iters);

/* One whole time step (Alg. 2): a1 + a2 if the factors are stale, const RHS, iterate until the stop rule holds, then
 * advance psi_{k+1/2} -> psi_{k-1/2} (a8) if advance != 0. Iterations are enqueued check_every at a time; every
 * iteration after the first of a batch looks at the residual of the one before it ON THE DEVICE and skips itself
 * once the rule held, so exactly the natural number of iterations runs; the host reads the residuals and the
 * executed-iterations counter once per batch (the only host round-trip).
 * iters_out[0] = iterations performed, iters_out[1] = iterations after which the rule first held (0 if never);
 * resid_out = last tested residual. Either may be NULL. [sync] up to the last residual read; the advance kernel may
 * still be in flight on the stream when the call returns (whatever the caller enqueues next on it is ordered after).
 * Returns > 0 (first singular cell, as oci_factor) when a1 + a2 ran inside this call and met a bad pivot: the factor is
 * enqueued together with the first batch of iterations, which then ran on zeroed inverses, so the call resets the
 * iterate to both time levels = psi_{k-1/2} (the state oci_set_state leaves; psi_{k-1/2}, q and the boundary data are
 * untouched), recomputes phi, empties the residual history and reports 0 iterations: a retry with another dt starts
 * from a defined state. */
int oci_step(oci_ctx *ctx, double tol, int32_t max_iters, int32_t check_every, int32_t stop_rule,
             int32_t advance, int32_t *iters_out, double *resid_out);

/* Source-iteration comparator (Alg. 1 / Appendix A): lagged scattering source, sweep each (g,m) through the
 * cells in the direction of mu_m (serial in space, parallel over angle x group), phi, residual. Same state,
 * same arguments and semantics as the OCI calls above. */
int si_iterate(oci_ctx *ctx, int32_t n_iters);
int si_step(oci_ctx *ctx, double tol, int32_t max_iters, int32_t check_every, int32_t stop_rule,
            int32_t advance, int32_t *iters_out, double *resid_out);

int oci_advance(oci_ctx *ctx);                                   /* a8 alone [async] */
int oci_scalar_flux(oci_ctx *ctx, double *phi_dev);              /* [J][G][4] of the current iterate [async] */
int oci_angular_flux(oci_ctx *ctx, double *psi_dev);             /* [J][G][N][4] current iterate [async]     */

/* Residuals of the last oci_step / si_step (or since the last one, for bare *_iterate calls):
 * kind 0 = max |dphi| per iteration, kind 1 = ||dPsi||_2 (OCI) or ||dphi||_2 (SI) per iteration (only
 * recorded under OCI_STOP_PAPER). host_out[cap]; *n = entries available. [sync] */
int oci_residual_history(oci_ctx *ctx, int32_t kind, double *host_out, int32_t cap, int32_t *n);

/* End-to-end convenience for host callers (bench.py's e2e leg): H2D of q_host [J][G][4] (NULL = keep),
 * oci_step or si_step (scheme 0 = OCI incl. oci_factor if stale, 1 = SI), D2H of phi into phi_host
 * [J][G][4]. Host buffers should be pinned for full copy bandwidth. [sync] */
int oci_step_host(oci_ctx *ctx, int32_t scheme, const double *q_host, double tol, int32_t max_iters,
                  int32_t check_every, int32_t stop_rule, int32_t advance, int32_t *iters_out,
                  double *resid_out, double *phi_host);

/* Debug / parity helpers (tests only). A_host, Ainv_host: [n][n] row-major. [sync] */
int oci_debug_get_matrix(oci_ctx *ctx, int32_t cell, double *A_host);   /* assembled, un-eliminated A_j  */
/* The same matrix as the PRODUCTION factor kernel selected by the current options assembles it on chip (a1 inside the
 * a1 + a2 launch), dumped before the elimination starts -- what the bit-exactness test of the production assembly
 * reads. OCI_E_UNSUPPORTED when that kernel assembles through the same device function as oci_debug_get_matrix
 * (the generic shared-memory kernel) or in solve_mode 1. */
int oci_debug_get_factor_input(oci_ctx *ctx, int32_t cell, double *A_host);
int oci_debug_get_inverse(oci_ctx *ctx, int32_t cell, double *Ainv_host);/* what oci_factor stored for j
                                                                          (OCI_E_UNSUPPORTED in solve_mode 1); also
                                                                          after an oci_factor that reported singular
                                                                          cells: zeros for those, A_j^{-1} elsewhere */
int oci_debug_get_const_rhs(oci_ctx *ctx, double *c_dev);               /* [J][n] c_j of a3 [async]       */

/* Enqueues `count` launches of an empty kernel (one CTA per SM) on the context's stream: the launch floor that the
 * per-iteration times of the L2-resident configurations (BASELINE.json configs 1-2) are quoted against. [async] */
int oci_debug_empty_launches(oci_ctx *ctx, int32_t count);

/* Device time (ms, CUDA events on the context's stream) of the most recent call of each kind:
 * which 0 = oci_factor, 1 = oci_iterate / the iterations inside oci_step, 2 = si_iterate / si_step iterations.
 * *launches = kernels launched by that call. [sync] */
int oci_last_timing(oci_ctx *ctx, int32_t which, double *ms, int64_t *launches);

/* ---- The one entry point that needs no allocation at all ------------------------------------------------------
 * Every call above works out of the workspace the caller allocated for oci_create. Some callers cannot allocate:
 * a transport module inside a host application whose memory manager owns the whole GPU and passes the module its
 * arrays but no allocator, or code on a path where cudaMalloc / cudaFree are off limits because they synchronise the
 * device and stall the process's other streams (a convergence monitor called between a coupled code's iterations).
 * For them: a6 + a7 (Eq. 44; the tested quantities of the stop rules, PAPER.md:166-171 and
 * BASELINE.json) on arrays the caller already has, with no context and no workspace:
 *     phi[j][g][p] = sum_m w[m] psi[j][g][m][p],   resid[0] = max |phi - phi_prev|,   resid[1] = ||phi - phi_prev||_2
 * (a NaN anywhere gives resid[0] = +inf, like the residual history). All five arrays are DEVICE pointers on one GPU,
 * fp64, layouts as at the top of this header; resid_dev holds 2 doubles; phi_dev may be the same array as
 * phi_prev_dev (update in place), no other overlap. [async] on cuda_stream (a cudaStream_t of that GPU, NULL = legacy
 * default stream); the arrays must stay alive until the stream has passed the call.
 *
 * The kernel's scratch (one partial result per CTA and a counter) lives in a static __device__ array inside the
 * library, OCI_STATIC_SCRATCH_BYTES on every GPU that loads liboci_b200.so, held until the process exits. The call
 * itself runs no cudaMalloc, cudaFree or any other allocating routine. Consequences the caller has to know:
 *  - Limit: J * G <= OCI_STATIC_MAX_PAIRS; anything larger returns OCI_E_TOO_LARGE and launches nothing.
 *  - The first call on each GPU looks up the array's device address (cudaGetSymbolAddress) and keeps it; make that
 *    first call before starting any stream capture on the thread.
 *  - All calls on one GPU share the array. Each call clears the counter it needs on its stream before its kernel, so
 *    calls that follow one another on a stream (or are otherwise ordered) are fine; two calls whose kernels can run on
 *    the GPU at the same time (different streams, different threads) race on it and give wrong residuals.
 * Returns 0, -i for a bad i-th argument (null, not device memory, or on another GPU than psi_dev), OCI_E_TOO_LARGE,
 * or OCI_E_CUDA (oci_static_last_cuda_error() has the cudaError_t of the calling thread's last such failure). */
#define OCI_STATIC_MAX_PAIRS (1 << 20)                               /* largest J * G (cells x groups)            */
#define OCI_STATIC_SCRATCH_BYTES (256 + (OCI_STATIC_MAX_PAIRS / 64) * 16) /* 262400 B of device memory per GPU    */
int oci_flux_residual_static(int32_t J, int32_t N, int32_t G, const double *w_dev, const double *psi_dev,
                             const double *phi_prev_dev, double *phi_dev, double *resid_dev, void *cuda_stream);
int oci_static_last_cuda_error(void);

#ifdef __cplusplus
}
#endif
#endif /* OCI_B200_H */
