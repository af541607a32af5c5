// vmg_noalloc.cu -- vmg_norm_inf_static: the maximum norm (S6; the norm of the exit rules, 8(c) C5 / R12)
// for callers that cannot allocate: no handle, no cudaMalloc / cudaFree, no allocating library routine, no
// synchronisation.  A variant of norm_inf_kernel (vmg_kernels.cuh), whose scratch is the handle's cudaMalloc'ed scalar
// block: here the scratch is a file-scope __device__ array that every GPU loading the library holds until exit.
//
// Self-contained on purpose: it includes none of the library's kernel headers (their __global__ functions are defined
// once, in vmg_api.cu) and changes no existing code path.
#include "../../include/vmg.h"

#include <cuda_runtime.h>
#include <mutex>

namespace {

constexpr int kThreads = 256;
constexpr int kPerThread = 16;
constexpr long long kChunk = (long long)kThreads * kPerThread;                  // elements per CTA: 4096
constexpr int kMaxBlocks = (int)(VMG_NORM_INF_STATIC_MAX_N / kChunk);           // 32 768 partial maxima
constexpr int kHeader = 32;                                                     // 256 bytes: [0] = the ticket counter
static_assert(VMG_NORM_INF_STATIC_MAX_N % kChunk == 0, "the limit is a whole number of chunks");

// The scratch: 256 B header + one partial maximum (bit pattern) per chunk = 262 400 bytes per GPU.
// HOST code must not pass this name to a kernel (there it is a host-side stand-in, not a device address):
// scratch_of_current_device() asks the runtime for the device address once per device.
static __device__ __align__(256) unsigned long long vmg_norm_static_scratch[kHeader + kMaxBlocks];

// |x| as a bit pattern; non-negative doubles order like unsigned integers, a NaN becomes the quiet-NaN pattern, which
// is larger than every finite value and +Inf (the convention of block_max_to_global / norm_inf_kernel)
__device__ __forceinline__ unsigned long long abs_bits(double x)
{
    double a = fabs(x);
    return a != a ? 0x7ff8000000000000ull : (unsigned long long)__double_as_longlong(a);
}

__device__ __forceinline__ unsigned long long block_max_bits(unsigned long long b)
{
    __shared__ unsigned long long warp_max[kThreads / 32];
    for (int o = 16; o > 0; o >>= 1) {
        unsigned long long other = __shfl_xor_sync(0xffffffffu, b, o);
        b = other > b ? other : b;
    }
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    __syncthreads();                                   // warp_max may still be read from the previous call
    if (lane == 0) warp_max[w] = b;
    __syncthreads();
    b = lane < kThreads / 32 ? warp_max[lane] : 0ull;
    for (int o = 16; o > 0; o >>= 1) {
        unsigned long long other = __shfl_xor_sync(0xffffffffu, b, o);
        b = other > b ? other : b;
    }
    return b;                                          // every thread of the block holds the block's maximum
}

// CTA b: maximum over its chunk -> scratch[kHeader + b]; the CTA that draws the last ticket reduces the partials of
// all CTAs and writes *out.  scratch[0] (the ticket counter) must be 0 at launch: the entry point clears it.
__global__ void __launch_bounds__(kThreads)
norm_inf_static_kernel(const double* __restrict__ v, long long n, unsigned long long* scratch, double* out)
{
    const long long base = (long long)blockIdx.x * kChunk;
    unsigned long long m = 0ull;
#pragma unroll
    for (int u = 0; u < kPerThread; ++u) {
        const long long t = base + threadIdx.x + (long long)u * kThreads;
        if (t < n) {
            const unsigned long long b = abs_bits(v[t]);
            m = b > m ? b : m;
        }
    }
    m = block_max_bits(m);
    __shared__ int last;
    if (threadIdx.x == 0) {
        scratch[kHeader + blockIdx.x] = m;
        __threadfence();                               // the partial before the ticket
        last = atomicAdd(&scratch[0], 1ull) == (unsigned long long)gridDim.x - 1ull;
    }
    __syncthreads();
    if (!last) return;
    __threadfence();
    m = 0ull;
    for (int b = threadIdx.x; b < (int)gridDim.x; b += kThreads) {
        const unsigned long long p = __ldcg(&scratch[kHeader + b]);   // written by other SMs: read at L2
        m = p > m ? p : m;
    }
    m = block_max_bits(m);
    if (threadIdx.x == 0) *out = __longlong_as_double((long long)m);
}

constexpr int kMaxDevices = 64;
std::mutex g_mutex;
unsigned long long* g_scratch[kMaxDevices] = {};

// device address of the scratch on the CURRENT device (cudaGetSymbolAddress once per device, with that device current)
cudaError_t scratch_of_current_device(unsigned long long** p)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_mutex);
    if (!g_scratch[dev]) {
        void* addr = nullptr;
        e = cudaGetSymbolAddress(&addr, vmg_norm_static_scratch);
        if (e != cudaSuccess) return e;
        g_scratch[dev] = (unsigned long long*)addr;
    }
    *p = g_scratch[dev];
    return cudaSuccess;
}

int fail(const char** why, int code, const char* text)
{
    if (why) *why = text;
    return code;
}

}  // namespace

extern "C" int vmg_norm_inf_static(const double* v, long long n, double* out, void* cuda_stream, const char** why)
{
    if (why) *why = "ok";
    if (!out) return fail(why, VMG_ERR_ARG, "vmg_norm_inf_static: out is NULL");
    if (n < 0) return fail(why, VMG_ERR_ARG, "vmg_norm_inf_static: n is negative");
    if (n > 0 && !v) return fail(why, VMG_ERR_ARG, "vmg_norm_inf_static: v is NULL");
    if (n > VMG_NORM_INF_STATIC_MAX_N)
        return fail(why, VMG_ERR_SIZE,
                    "vmg_norm_inf_static: n exceeds VMG_NORM_INF_STATIC_MAX_N = 134217728 doubles (the static scratch holds "
                    "one partial maximum per 4096 elements); use vmg_step_norm_inf or split the array");
    unsigned long long* scratch = nullptr;
    if (scratch_of_current_device(&scratch) != cudaSuccess) {
        (void)cudaGetLastError();
        return fail(why, VMG_ERR_CUDA, "vmg_norm_inf_static: cudaGetSymbolAddress of the static scratch failed");
    }
    cudaStream_t stream = (cudaStream_t)cuda_stream;
    // the ticket counter must start at zero; the partials need no clearing (every entry read is written first)
    if (cudaMemsetAsync(scratch, 0, sizeof(unsigned long long), stream) != cudaSuccess) {
        (void)cudaGetLastError();
        return fail(why, VMG_ERR_CUDA, "vmg_norm_inf_static: cudaMemsetAsync of the ticket counter failed");
    }
    const unsigned blocks = n > 0 ? (unsigned)((n + kChunk - 1) / kChunk) : 1u;
    norm_inf_static_kernel<<<blocks, kThreads, 0, stream>>>(v, n, scratch, out);
    if (cudaGetLastError() != cudaSuccess)
        return fail(why, VMG_ERR_CUDA, "vmg_norm_inf_static: kernel launch failed");
    return VMG_OK;
}
