// dg_noalloc.cu -- dg_max_wavespeed_noalloc (include/dg_b200.h): the max-wavespeed reduction of DESIGN.md reading R10
// for callers that have no way of getting device memory for the library.
//
// Who that is.  Everything else in this library works out of a workspace the caller allocates once and hands to
// dg_bind.  Some callers cannot do even that: a monitoring or time-step-control hook that a host application calls
// from inside its time loop with nothing but a pointer to the solution and a slot for the answer; a plug-in that
// runs under an application which has handed out all device memory up front and treats any later cudaMalloc as a bug
// (it synchronises the whole device, it can fail half-way through a run on a fragmented or full card, and its
// pool may be private to the application); code on a path where an allocation failure cannot be reported upwards.
// For them the reduction's scratch memory lives in THIS FILE, in a file-scope __device__ array of fixed size that the
// CUDA runtime places on every GPU that loads the library and keeps there until the process exits.
//
// The kernel is the stand-alone dg_wavespeed_kernel of dg_kernels.cu with two changes: it reads the state in the
// canonical layout (the caller has no context, so there is no internal layout), and instead of one 64-bit atomicMax
// per warp on a workspace word it keeps one partial maximum per thread block in the static array; the block that
// finishes last folds the partials into the caller's output.  Node arithmetic and NaN rule are the same, and the
// maximum is taken on the bit patterns exactly as atomicMax does there, so both paths give the same double.
//
// Shares no state with dg_api.cu / dg_kernels.cu and changes none of their code paths.
#include <cuda_runtime.h>

#include <cstdarg>
#include <cstdio>
#include <mutex>

#include "../../include/dg_b200.h"

namespace {

constexpr int kThreads = 256;                       // threads per block
constexpr int kNodesPerThread = 64;
constexpr size_t kTile = (size_t)kThreads * kNodesPerThread;                    // 16,384 nodes per thread block
constexpr size_t kMaxBlocks = (size_t)DG_NOALLOC_MAX_NODES / kTile;             // 32,768 partial maxima
constexpr size_t kHead = 32;                        // the first 256 bytes: word 0 = count of finished blocks
static_assert(kMaxBlocks * kTile == (size_t)DG_NOALLOC_MAX_NODES, "DG_NOALLOC_MAX_NODES must be a whole number of tiles");

// THE scratch memory: 256 B + 8 B per block = 256.25 KiB on every GPU that loads libdg_b200.so, until exit.
// In host code this name is only a handle for cudaGetSymbolAddress: it is NOT a device address and must never be
// passed to a kernel (scratch_of_current_device() below turns it into one).  Device code may name it directly.
static __device__ __align__(256) unsigned long long g_noalloc_scratch[kHead + kMaxBlocks];

__global__ void __launch_bounds__(kThreads) dg_wavespeed_noalloc_kernel(const double *__restrict__ q, size_t n_nodes,
                                                                        double gamma, double gm1,
                                                                        unsigned long long *scratch, double *lam_out) {
    __shared__ unsigned long long warp_best[kThreads / 32];
    __shared__ bool last_block;
    const size_t base = (size_t)blockIdx.x * kTile;
    double best = 0.0;
    for (int it = 0; it < kNodesPerThread; ++it) {
        const size_t node = base + (size_t)it * kThreads + threadIdx.x;
        if (node >= n_nodes) break;
        const double *qn = q + node * 5;             // canonical layout: the five variables of a node are adjacent
        const double Q0 = qn[0], Q1 = qn[1], Q2 = qn[2], Q3 = qn[3], Q4 = qn[4];
        const double rinv = 1.0 / Q0;
        const double u = Q1 * rinv, v = Q2 * rinv, w = Q3 * rinv;
        const double pres = gm1 * (Q4 - 0.5 * Q0 * (u * u + v * v + w * w));
        const double s = sqrt(u * u + v * v + w * w) + sqrt(gamma * pres * rinv);
        if (s > best || s != s) best = s;            // NaN sticks (reading R15)
    }
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
        const double o = __shfl_xor_sync(0xffffffffu, best, off);
        if (o > best || o != o) best = o;
    }
    // from here on the maximum is taken on the bit patterns, as the atomicMax of the workspace path does:
    // non-negative doubles order like integers and every NaN pattern lies above them
    if ((threadIdx.x & 31) == 0) warp_best[threadIdx.x >> 5] = (unsigned long long)__double_as_longlong(best);
    __syncthreads();
    if (threadIdx.x == 0) {
        unsigned long long b = warp_best[0];
        for (int i = 1; i < kThreads / 32; ++i) b = warp_best[i] > b ? warp_best[i] : b;
        scratch[kHead + blockIdx.x] = b;
        __threadfence();                              // the partial is visible before the count moves
        last_block = atomicAdd(&scratch[0], 1ull) == (unsigned long long)gridDim.x - 1ull;
    }
    __syncthreads();
    if (!last_block) return;
    __threadfence();
    unsigned long long b = 0ull;
    for (unsigned i = threadIdx.x; i < gridDim.x; i += kThreads) {
        const unsigned long long o = __ldcg(&scratch[kHead + i]);   // written by other blocks: read past L1
        b = o > b ? o : b;
    }
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
        const unsigned long long o = __shfl_xor_sync(0xffffffffu, b, off);
        b = o > b ? o : b;
    }
    if ((threadIdx.x & 31) == 0) warp_best[threadIdx.x >> 5] = b;
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int i = 0; i < kThreads / 32; ++i) b = warp_best[i] > b ? warp_best[i] : b;
        *lam_out = __longlong_as_double((long long)b);
        scratch[0] = 0ull;                            // leave the count as the next call needs it
    }
}

// Set-up, once per device: ask the runtime where ITS copy of g_noalloc_scratch lives on the current device.
constexpr int kMaxDevices = 64;
std::mutex g_setup_mutex;
unsigned long long *g_scratch_of_device[kMaxDevices] = {};

cudaError_t scratch_of_current_device(unsigned long long **out, int *device) {
    cudaError_t e = cudaGetDevice(device);
    if (e != cudaSuccess) return e;
    if (*device < 0 || *device >= kMaxDevices) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_setup_mutex);
    if (!g_scratch_of_device[*device]) {
        void *p = nullptr;
        e = cudaGetSymbolAddress(&p, g_noalloc_scratch);
        if (e != cudaSuccess) return e;
        if (!p) return cudaErrorInvalidSymbol;
        g_scratch_of_device[*device] = static_cast<unsigned long long *>(p);
    }
    *out = g_scratch_of_device[*device];
    return cudaSuccess;
}

int fail(char *err, size_t err_len, int code, const char *fmt, ...) {
    if (err && err_len) {
        va_list ap;
        va_start(ap, fmt);
        std::vsnprintf(err, err_len, fmt, ap);
        va_end(ap);
    }
    return code;
}

}  // namespace

extern "C" int dg_max_wavespeed_noalloc(const double *q_dev, size_t n_nodes, double gamma, double *lam_out_dev,
                                        void *cuda_stream, char *err, size_t err_len) {
    if (err && err_len) err[0] = '\0';
    // argument checks first: they touch no GPU
    if (!q_dev || !lam_out_dev) return fail(err, err_len, DG_EINVAL, "dg_max_wavespeed_noalloc: null pointer");
    if (!(gamma > 1.0)) return fail(err, err_len, DG_EINVAL, "dg_max_wavespeed_noalloc: gamma = %g must be > 1", gamma);
    if (n_nodes == 0) return fail(err, err_len, DG_EINVAL, "dg_max_wavespeed_noalloc: n_nodes = 0");
    if (n_nodes > (size_t)DG_NOALLOC_MAX_NODES)
        return fail(err, err_len, DG_ENOMEM,
                    "dg_max_wavespeed_noalloc: n_nodes = %zu is beyond DG_NOALLOC_MAX_NODES = %zu, the most the fixed "
                    "scratch array holds (this call never allocates; use dg_bind + dg_max_wavespeed for larger states)",
                    n_nodes, (size_t)DG_NOALLOC_MAX_NODES);
    unsigned long long *scratch = nullptr;
    int device = -1;
    cudaError_t e = scratch_of_current_device(&scratch, &device);
    if (e != cudaSuccess)
        return fail(err, err_len, DG_ECUDA, "dg_max_wavespeed_noalloc: cudaGetSymbolAddress on device %d: %s", device,
                    cudaGetErrorString(e));
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    // the array keeps whatever the last call (or a call that was cut short) left: the count must start at zero;
    // the partial maxima need no clearing, every block of this launch overwrites its own before any is read
    e = cudaMemsetAsync(scratch, 0, kHead * sizeof(unsigned long long), stream);
    if (e != cudaSuccess)
        return fail(err, err_len, DG_ECUDA, "dg_max_wavespeed_noalloc: clearing the scratch head: %s", cudaGetErrorString(e));
    const unsigned blocks = (unsigned)((n_nodes + kTile - 1) / kTile);
    dg_wavespeed_noalloc_kernel<<<blocks, kThreads, 0, stream>>>(q_dev, n_nodes, gamma, gamma - 1.0, scratch, lam_out_dev);
    e = cudaGetLastError();
    if (e != cudaSuccess)
        return fail(err, err_len, DG_ECUDA, "dg_max_wavespeed_noalloc: kernel launch: %s", cudaGetErrorString(e));
    return DG_OK;
}
