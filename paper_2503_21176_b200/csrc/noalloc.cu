// noalloc.cu -- sqeq_energy_noalloc: E = 1/2 sum_i q_i phi_i (Eq. 5) without any allocation.
//
// For callers that cannot call cudaMalloc (code under CUDA-graph capture, tight serving loops, harnesses that forbid
// it).  The library's own path forms this sum inside k_assemble with fp64 atomics into a cudaMalloc'ed context
// workspace (sqeq_create allocates).  This variant is a two-stage reduction whose scratch -- one fp64 partial sum per
// block and the counter that elects the last block -- lives in a file-scope __device__ array: every GPU that loads the
// library holds its 32.25 KB until the process exits.  Limit: SQEQ_NOALLOC_MAX_N atoms.
//
// The array's name is a HOST-side stand-in in host code, not a device address; the device address comes from
// cudaGetSymbolAddress, once per device, with that device current (noalloc_setup below), and is what the kernel gets.
// Every call on a device shares the array: calls that overlap on the GPU (two streams) race; calls on one stream are
// ordered and safe.  The counter must start at zero: it is cleared on the stream before every launch and reset by the
// electing block; the partial sums need no clearing (every slot read is written by the same launch).
// The summation order is fixed (no floating-point atomics): the same inputs give the same bits on every call.
#include "common.cuh"
#include <mutex>

#define NA_CHUNK 1024                                        // elements per block
#define NA_MAX_BLOCKS 4096
static_assert((int64_t)NA_CHUNK * NA_MAX_BLOCKS == SQEQ_NOALLOC_MAX_N, "include/sqeq.h states the limit");

struct NaScratch {
    double partial[NA_MAX_BLOCKS];
    unsigned done;                                           // blocks that have written their partial sum
    unsigned pad[63];
};
static __device__ __align__(256) NaScratch g_na_scratch;

__device__ __forceinline__ double na_block_sum(double v, double* red)          // 256 threads; result in thread 0
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = v;
    __syncthreads();
    if (threadIdx.x < 8) {
        v = red[threadIdx.x];
#pragma unroll
        for (int o = 4; o > 0; o >>= 1) v += __shfl_xor_sync(0xffu, v, o);
    }
    __syncthreads();
    return v;
}

__global__ void __launch_bounds__(256)
k_energy_noalloc(int64_t n, const float* __restrict__ q, const float* __restrict__ phi, NaScratch* s, double* __restrict__ out)
{
    __shared__ double red[8];
    __shared__ bool last;
    const int64_t beg = (int64_t)blockIdx.x * NA_CHUNK;
    const int64_t end = beg + NA_CHUNK < n ? beg + NA_CHUNK : n;
    double v = 0.0;
    for (int64_t i = beg + threadIdx.x; i < end; i += 256) v += (double)q[i] * (double)phi[i];
    v = na_block_sum(v, red);
    if (threadIdx.x == 0) {
        s->partial[blockIdx.x] = v;
        __threadfence();                                     // the partial sum before the count
        last = atomicAdd(&s->done, 1u) == gridDim.x - 1;
    }
    __syncthreads();
    if (!last) return;
    __threadfence();
    double t = 0.0;
    for (unsigned b = threadIdx.x; b < gridDim.x; b += 256) t += ((volatile double*)s->partial)[b];
    t = na_block_sum(t, red);
    if (threadIdx.x == 0) {
        *out = 0.5 * t;
        s->done = 0;                                         // as the next call must find it
    }
}

// ---- host side --------------------------------------------------------------------------------------------------
#define NA_MAX_DEVICES 64
static std::mutex g_na_mutex;
static NaScratch* g_na_ptr[NA_MAX_DEVICES];                  // device address of g_na_scratch, per device

// Once per device, with that device current: the device address of the scratch array.
static int noalloc_setup(int device, NaScratch** out)
{
    std::lock_guard<std::mutex> lock(g_na_mutex);
    if (!g_na_ptr[device]) {
        NaScratch* p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress((void**)&p, g_na_scratch);
        if (e != cudaSuccess || !p) {
            cudaGetLastError();
            return sqeq_fail(nullptr, SQEQ_ECUDA, "sqeq_energy_noalloc: cudaGetSymbolAddress on device %d failed: %s", device,
                             cudaGetErrorString(e));
        }
        g_na_ptr[device] = p;
    }
    *out = g_na_ptr[device];
    return SQEQ_OK;
}

extern "C" int sqeq_energy_noalloc(int device, void* cuda_stream, int64_t n, const float* q, const float* phi,
                                   double* energy_dev)
{
    if (device < 0 || device >= NA_MAX_DEVICES)
        return sqeq_fail(nullptr, SQEQ_EINVAL, "sqeq_energy_noalloc: device %d out of range [0, %d)", device, NA_MAX_DEVICES);
    if (n < 1 || n > (int64_t)SQEQ_NOALLOC_MAX_N)
        return sqeq_fail(nullptr, SQEQ_EINVAL, "sqeq_energy_noalloc: n = %lld outside [1, %lld] (the static scratch array holds "
                                               "one partial sum per %d atoms, %d of them)",
                         (long long)n, (long long)SQEQ_NOALLOC_MAX_N, NA_CHUNK, NA_MAX_BLOCKS);
    if (!q || !phi || !energy_dev) return sqeq_fail(nullptr, SQEQ_EINVAL, "sqeq_energy_noalloc: NULL argument");
    cudaError_t e = cudaSetDevice(device);
    if (e != cudaSuccess) {
        cudaGetLastError();
        return sqeq_fail(nullptr, SQEQ_ECUDA, "sqeq_energy_noalloc: cudaSetDevice(%d): %s", device, cudaGetErrorString(e));
    }
    NaScratch* s = nullptr;
    SQEQ_TRY(noalloc_setup(device, &s));
    cudaStream_t st = (cudaStream_t)cuda_stream;
    e = cudaMemsetAsync(&s->done, 0, sizeof(unsigned), st);  // device address arithmetic on the host: no dereference
    if (e == cudaSuccess) {
        const int nb = (int)((n + NA_CHUNK - 1) / NA_CHUNK);
        k_energy_noalloc<<<nb, 256, 0, st>>>(n, q, phi, s, energy_dev);
        e = cudaGetLastError();
    }
    if (e != cudaSuccess)
        return sqeq_fail(nullptr, SQEQ_ECUDA, "sqeq_energy_noalloc: launch failed: %s", cudaGetErrorString(e));
    return SQEQ_OK;
}
