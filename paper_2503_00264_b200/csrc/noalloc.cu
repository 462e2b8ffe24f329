// noalloc.cu -- oci_flux_residual_static (include/oci.h): a6 + a7 for arrays the caller already holds, with no
// device-memory allocation anywhere on the path.
//
// Who needs it. Everything else in this library works out of one workspace that the caller allocates up front
// (oci_workspace_bytes -> cudaMalloc / torch.empty -> oci_create). Two kinds of caller cannot do that:
//   * a transport module embedded in a host application whose own memory manager has claimed the GPU's memory and
//     hands the module a fixed set of device arrays (psi, phi) but no allocator: there is nothing left for a
//     cudaMalloc to return, and no handle to ask the host for more;
//   * a caller on a path where cudaMalloc / cudaFree are ruled out because they synchronise the whole device and stall
//     every other stream of the process -- e.g. a convergence monitor that a coupled code calls between two of its own
//     iterations, on arrays it has anyway.
// For them this file keeps the scratch the kernel needs in a file-scope __device__ array: it is part of the loaded
// module, so every GPU that loads liboci_b200.so holds OCI_STATIC_SCRATCH_BYTES (262400 B, about 256 KB) of it until
// the process exits, and no call ever allocates.
//
// What the kernel does is what the tail of every iterate kernel does (iterate.cu, si.cu si_finish_kernel):
// phi = sum_m w_m psi_m (Eq. 44) and the two residuals of the stop rules, max |dphi| (BASELINE.json's
// rule) and ||dphi||_2 (Eq. 13, as the SI loop of Alg. 1 uses it). Those kernels accumulate the
// residual with atomics into workspace slots that reset_history() zeroes; here every CTA writes its partial result
// into its own slot of the static array and the CTA that finishes last combines the slots in index order, so the
// result does not depend on the order in which the CTAs ran.
#include "common.cuh"
#include <mutex>

namespace {

constexpr int NA_THREADS = 256;                                             // one thread per entry (j, g, p) of phi
constexpr int NA_PAIRS_PER_CTA = NA_THREADS / 4;
constexpr int NA_MAX_CTAS = OCI_STATIC_MAX_PAIRS / NA_PAIRS_PER_CTA;        // 16384
constexpr size_t NA_HEADER = 256;                                           // [0] = CTAs finished (must start at 0)
static_assert(NA_HEADER + (size_t)NA_MAX_CTAS * sizeof(double2) == OCI_STATIC_SCRATCH_BYTES, "oci.h out of step");

// The scratch. In HOST code this name is only a handle for cudaGetSymbolAddress (its host-side address is not device
// memory); the kernel below is always given the device address looked up in scratch_of().
static __device__ __align__(256) unsigned char g_static_scratch[OCI_STATIC_SCRATCH_BYTES];

__global__ void __launch_bounds__(NA_THREADS)
flux_residual_static_kernel(size_t total, int N, const double *__restrict__ w, const double *__restrict__ psi,
                            const double *phi_prev, double *phi, double *__restrict__ resid,
                            unsigned char *scratch)
{
    __shared__ double s_max[NA_THREADS / 32], s_sum[NA_THREADS / 32];
    __shared__ bool s_last;
    unsigned int *finished = reinterpret_cast<unsigned int *>(scratch);
    double2 *partial = reinterpret_cast<double2 *>(scratch + NA_HEADER);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const size_t e = (size_t)blockIdx.x * NA_THREADS + tid;
    double ad = 0.0, sq = 0.0;
    if (e < total) {
        const int p = (int)(e & 3);
        const size_t jg = e >> 2;
        double s = 0.0;
        for (int m = 0; m < N; ++m) s = fma(w[m], psi[(jg * N + m) * 4 + p], s); // same order as scalar_flux_kernel
        const double d = s - phi_prev[e]; // phi may be phi_prev: entry e is read here and written below, by this thread only
        phi[e] = s;
        ad = fabs(d);
        sq = d * d;
    }
    ad = warp_max(ad);
    sq = warp_sum(sq);
    if (lane == 0) { s_max[warp] = ad; s_sum[warp] = sq; }
    __syncthreads();
    if (tid == 0) {
        double mx = s_max[0], sm = s_sum[0];
        for (int i = 1; i < NA_THREADS / 32; ++i) {
            mx = (s_max[i] > mx || !(s_max[i] == s_max[i])) ? s_max[i] : mx;
            sm += s_sum[i];
        }
        partial[blockIdx.x] = make_double2(mx, sm);
        __threadfence(); // the slot is visible device-wide before this CTA counts itself as finished
        s_last = atomicAdd(finished, 1u) == gridDim.x - 1;
    }
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    // last CTA: every slot 0 .. gridDim.x - 1 of THIS call is complete (slots beyond it still hold older calls' values
    // and are not read). Thread t folds slots t, t + 256, ... in that order, then the 256 results fold in thread order.
    double mx = 0.0, sm = 0.0;
    for (unsigned int b = tid; b < gridDim.x; b += NA_THREADS) {
        const double2 v = __ldcg(partial + b);
        mx = (v.x > mx || !(v.x == v.x)) ? v.x : mx;
        sm += v.y;
    }
    mx = warp_max(mx);
    sm = warp_sum(sm);
    __syncthreads();
    if (lane == 0) { s_max[warp] = mx; s_sum[warp] = sm; }
    __syncthreads();
    if (tid == 0) {
        mx = s_max[0]; sm = s_sum[0];
        for (int i = 1; i < NA_THREADS / 32; ++i) {
            mx = (s_max[i] > mx || !(s_max[i] == s_max[i])) ? s_max[i] : mx;
            sm += s_sum[i];
        }
        if (!(mx == mx)) mx = __longlong_as_double(0x7ff0000000000000LL); // NaN reported as +inf, as resid_bits() does
        resid[0] = mx;
        resid[1] = sqrt(sm);
    }
}

// Device address of g_static_scratch on device `dev`, looked up once per device with that device current.
constexpr int NA_MAX_DEVICES = 64;
std::mutex g_lock;
unsigned char *g_scratch_dev[NA_MAX_DEVICES];

cudaError_t scratch_of(int dev, unsigned char **out)
{
    std::lock_guard<std::mutex> hold(g_lock);
    if (!g_scratch_dev[dev]) {
        void *p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(&p, g_static_scratch); // `dev` is current (DeviceGuard in the caller)
        if (e != cudaSuccess) return e;
        g_scratch_dev[dev] = static_cast<unsigned char *>(p);
    }
    *out = g_scratch_dev[dev];
    return cudaSuccess;
}

thread_local int g_static_cuda_error = 0;

int cuda_fail(cudaError_t e)
{
    g_static_cuda_error = (int)e;
    (void)cudaGetLastError();
    return OCI_E_CUDA;
}

// device that owns `p`, or -1 if `p` is not device (or managed) memory
int device_of(const void *p)
{
    cudaPointerAttributes pa;
    if (cudaPointerGetAttributes(&pa, p) != cudaSuccess) { (void)cudaGetLastError(); return -1; }
    if (pa.type != cudaMemoryTypeDevice && pa.type != cudaMemoryTypeManaged) return -1;
    return pa.device;
}

} // namespace

extern "C" {

int oci_flux_residual_static(int32_t J, int32_t N, int32_t G, const double *w_dev, const double *psi_dev,
                             const double *phi_prev_dev, double *phi_dev, double *resid_dev, void *cuda_stream)
{
    g_static_cuda_error = 0;
    if (J < 1) return -1;
    if (N < 1) return -2;
    if (G < 1) return -3;
    if ((long long)J * G > OCI_STATIC_MAX_PAIRS) return OCI_E_TOO_LARGE; // before any CUDA call: testable without a GPU
    if (!w_dev) return -4;
    if (!psi_dev) return -5;
    if (!phi_prev_dev) return -6;
    if (!phi_dev) return -7;
    if (!resid_dev) return -8;
    const int dev = device_of(psi_dev);
    if (dev < 0 || dev >= NA_MAX_DEVICES) return -5;
    if (device_of(w_dev) != dev) return -4;
    if (device_of(phi_prev_dev) != dev) return -6;
    if (device_of(phi_dev) != dev) return -7;
    if (device_of(resid_dev) != dev) return -8;
    DeviceGuard guard(dev);
    unsigned char *scratch = nullptr;
    cudaError_t e = scratch_of(dev, &scratch);
    if (e != cudaSuccess) return cuda_fail(e);
    cudaStream_t stream = (cudaStream_t)cuda_stream;
    const size_t total = (size_t)J * G * 4;
    const unsigned int grid = (unsigned int)((total + NA_THREADS - 1) / NA_THREADS); // <= NA_MAX_CTAS by the size check
    // the finished-CTA counter must start at zero whatever the previous call (or a call that failed half-way) left
    e = cudaMemsetAsync(scratch, 0, NA_HEADER, stream);
    if (e != cudaSuccess) return cuda_fail(e);
    flux_residual_static_kernel<<<grid, NA_THREADS, 0, stream>>>(total, N, w_dev, psi_dev, phi_prev_dev, phi_dev, resid_dev,
                                                                 scratch);
    e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(e);
    return 0;
}

int oci_static_last_cuda_error(void) { return g_static_cuda_error; }

} // extern "C"
