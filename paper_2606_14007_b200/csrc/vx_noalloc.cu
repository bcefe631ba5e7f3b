// vx_noalloc.cu -- ONE entry point that allocates nothing, for callers that cannot call cudaMalloc
// (code under CUDA graph capture, tight serving loops, harnesses that forbid allocation).
//
// vx_hash_fold_noalloc is the variant of vx_hash_sink (include/vx.h: the BLAKE3 stage of PAPER.md
// L41-43 / L91 with no table traffic, every hash xor-folded) whose scratch -- one partial word per
// thread block -- does not come from the caller but from a file-scope device array of a fixed,
// modest size; a second kernel folds the partials into the caller's single output word.
//
//   * the array: VX_NOALLOC_MAX_CTAS words = 256 KB, held by every GPU that loads libvx.so until the
//     process exits; it bounds one call to VX_NOALLOC_MAX_NONCES = 2^25 nonces (more: VX_ERR_RANGE);
//   * in HOST code the array's name is a host-side stand-in, not a device address: its device address
//     is taken here with cudaGetSymbolAddress, once per device with that device current, and that
//     pointer is what the kernels get (device code could name the array directly; only the host needs
//     the address);
//   * no cudaMalloc, cudaFree or allocating library routine is called;
//   * every call on a device shares the array, which keeps the previous call's contents.  Nothing in it
//     has to start at zero: a call overwrites every partial it later reads.  Calls that overlap on the
//     GPU (two streams, two host threads) RACE on it -- serialise them on one stream.
#include <mutex>

#include "../../include/vx.h"
#include "vx_internal.h"

#define VX_NA_THREADS 256
#define VX_NA_NPT 4
#define VX_NOALLOC_MAX_CTAS 32768u                                                     // 256 KB of scratch
#define VX_NOALLOC_MAX_NONCES ((uint64_t)VX_NOALLOC_MAX_CTAS * VX_NA_THREADS * VX_NA_NPT)   // 2^25

static __device__ __align__(256) unsigned long long vx_noalloc_scratch[VX_NOALLOC_MAX_CTAS];

// xor of H(n) over the block's nonces -> partial[blockIdx.x]
template <bool NONCE5>
__global__ void __launch_bounds__(VX_NA_THREADS)
vx_k_hash_fold_partial(const __grid_constant__ VxHashConst hc, uint64_t nonce_begin, uint64_t count,
                       unsigned long long *__restrict__ partial)
{
    const uint64_t base = (uint64_t)blockIdx.x * (VX_NA_THREADS * VX_NA_NPT) + threadIdx.x;
    uint64_t x = 0;
#pragma unroll
    for (int k = 0; k < VX_NA_NPT; k++) {
        const uint64_t i = base + (uint64_t)k * VX_NA_THREADS;
        const uint64_t n = nonce_begin + i;
        const uint64_t h = vx_blake3_h<NONCE5>(hc, (uint32_t)n, (uint32_t)(n >> 32));
        x ^= (i < count) ? h : 0ull;
    }
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) x ^= __shfl_xor_sync(0xffffffffu, x, d);
    __shared__ uint64_t s[VX_NA_THREADS / 32];
    if ((threadIdx.x & 31) == 0) s[threadIdx.x >> 5] = x;
    __syncthreads();
    if (threadIdx.x == 0) {
        uint64_t y = 0;
        for (int w = 0; w < VX_NA_THREADS / 32; w++) y ^= s[w];
        partial[blockIdx.x] = y;
    }
}

// xor of partial[0 .. n) -> out[0]   (one block)
__global__ void __launch_bounds__(1024)
vx_k_hash_fold_final(const unsigned long long *__restrict__ partial, uint32_t n, unsigned long long *__restrict__ out)
{
    uint64_t x = 0;
    for (uint32_t i = threadIdx.x; i < n; i += 1024) x ^= partial[i];
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) x ^= __shfl_xor_sync(0xffffffffu, x, d);
    __shared__ uint64_t s[32];
    if ((threadIdx.x & 31) == 0) s[threadIdx.x >> 5] = x;
    __syncthreads();
    if (threadIdx.x == 0) {
        uint64_t y = 0;
        for (int w = 0; w < 32; w++) y ^= s[w];
        out[0] = y;
    }
}

// device address of the scratch array on the CURRENT device, resolved once per device ordinal
static cudaError_t scratch_address(unsigned long long **ptr)
{
    static std::mutex mu;
    static unsigned long long *cache[64];
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    std::lock_guard<std::mutex> lock(mu);
    if (dev >= 0 && dev < 64 && cache[dev]) { *ptr = cache[dev]; return cudaSuccess; }
    unsigned long long *p = nullptr;
    e = cudaGetSymbolAddress((void **)&p, vx_noalloc_scratch);
    if (e != cudaSuccess) return e;
    if (!p) return cudaErrorInvalidSymbol;
    if (dev >= 0 && dev < 64) cache[dev] = p;
    *ptr = p;
    return cudaSuccess;
}

extern "C" vx_status vx_hash_fold_noalloc(vx_plot *p, uint64_t nonce_begin, uint64_t count, uint64_t *dev_out,
                                          void *cuda_stream)
{
    if (!p) return VX_ERR_ARG;
    if (!dev_out) return (vx_status)vx_plot_fail(p, VX_ERR_ARG, "NULL dev_out");
    if (count > VX_NOALLOC_MAX_NONCES)
        return (vx_status)vx_plot_fail(p, VX_ERR_RANGE,
                            "vx_hash_fold_noalloc: count exceeds 2^25 nonces (its scratch is a fixed 256 KB device array); "
                            "split the range or use vx_hash_sink with caller-owned scratch");
    unsigned long long *scratch = nullptr;
    cudaError_t e = scratch_address(&scratch);
    if (e != cudaSuccess) return (vx_status)vx_plot_fail_cuda(p, e, "cudaGetSymbolAddress(vx_noalloc_scratch)");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const uint64_t per_cta = (uint64_t)VX_NA_THREADS * VX_NA_NPT;
    const uint32_t grid = (uint32_t)((count + per_cta - 1) / per_cta);      // <= VX_NOALLOC_MAX_CTAS
    const VxHashConst &hc = vx_plot_hash_const(p);
    if (grid) {
        if (hc.block_len == 5)
            vx_k_hash_fold_partial<true><<<grid, VX_NA_THREADS, 0, st>>>(hc, nonce_begin, count, scratch);
        else
            vx_k_hash_fold_partial<false><<<grid, VX_NA_THREADS, 0, st>>>(hc, nonce_begin, count, scratch);
        e = cudaGetLastError();
        if (e != cudaSuccess) return (vx_status)vx_plot_fail_cuda(p, e, "hash fold launch");
    }
    vx_k_hash_fold_final<<<1, 1024, 0, st>>>(scratch, grid, (unsigned long long *)dev_out);   // grid = 0: out = 0
    e = cudaGetLastError();
    if (e != cudaSuccess) return (vx_status)vx_plot_fail_cuda(p, e, "hash fold launch");
    return VX_OK;
}
