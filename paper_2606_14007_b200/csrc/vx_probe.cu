// vx_probe.cu -- measurement aid: dependent-free instruction chains that fix the issue rate of the
// SM's integer pipes, the denominator of stage 1's roofline ("The peak itself
// (lanes/clk/SM for LOP3, SHF, IADD3, IMAD on sm_100) is not in MEASURED_PEAKS.json -- measure it
// first with dependent-free instruction-chain microbenchmarks").  Not on the plot path.
//
// Every thread runs VX_PROBE_CHAINS independent chains of one instruction kind (each instruction
// depends only on the previous one of its own chain), 2048 threads per SM, so the pipe under test
// is the only limit.  bench.py --probe-alu times the launches with CUDA events and reports
// lane-ops per clock per SM; profiles/ holds the summary and the SASS opcode histogram of these
// kernels (what ptxas actually emitted for each kind).
#include "../../include/vx.h"
#include "vx_internal.h"

#define VX_PROBE_CHAINS 8
#define VX_PROBE_UNROLL 8      // instructions per chain per loop iteration
#define VX_PROBE_THREADS 256

template <int KIND>
__global__ void __launch_bounds__(VX_PROBE_THREADS)
vx_k_probe(uint32_t iters, uint32_t seed, uint32_t *__restrict__ out)
{
    uint32_t a[VX_PROBE_CHAINS];
    const uint32_t t = blockIdx.x * VX_PROBE_THREADS + threadIdx.x;
    uint32_t b = t * 0x9E3779B9u + seed, c = (t ^ seed) * 0x85EBCA6Bu + 1u;
#pragma unroll
    for (int k = 0; k < VX_PROBE_CHAINS; k++) a[k] = t + 0x01000193u * (k + 1);
    for (uint32_t i = 0; i < iters; i++) {
#pragma unroll
        for (int u = 0; u < VX_PROBE_UNROLL; u++) {
#pragma unroll
            for (int k = 0; k < VX_PROBE_CHAINS; k++) {
                if (KIND == VX_PROBE_LOP3)        // a = a ^ b ^ c : one LOP3
                    asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(a[k]) : "r"(b), "r"(c));
                else if (KIND == VX_PROBE_SHF)    // rotate right by 7 : one SHF.R.W
                    asm volatile("shf.r.wrap.b32 %0, %0, %0, 7;" : "+r"(a[k]));
                else if (KIND == VX_PROBE_ADD)    // 32-bit add; ptxas chooses IADD3 (ALU pipe) or IMAD.IADD (FMA pipe)
                    asm volatile("add.u32 %0, %0, %1;" : "+r"(a[k]) : "r"(b));
                else if (KIND == VX_PROBE_IMAD)   // a = a * b + c : IMAD (FMA pipe)
                    asm volatile("mad.lo.u32 %0, %0, %1, %2;" : "+r"(a[k]) : "r"(b), "r"(c));
                else if (KIND == VX_PROBE_PRMT)   // byte permute : PRMT
                    asm volatile("prmt.b32 %0, %0, %1, 0x0321;" : "+r"(a[k]) : "r"(b));
                else {                            // VX_PROBE_ARX: BLAKE3's mix, xor then rotate (LOP3 + SHF) per 2 ops
                    if (u & 1) asm volatile("shf.r.wrap.b32 %0, %0, %0, 12;" : "+r"(a[k]));
                    else asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(a[k]) : "r"(b), "r"(c));
                }
            }
        }
    }
    uint32_t x = 0;
#pragma unroll
    for (int k = 0; k < VX_PROBE_CHAINS; k++) x ^= a[k];
    if (x == 0x5bd1e995u) out[t & 1023u] = x;    // keeps the chains alive; practically never taken
}

extern "C" vx_status vx_probe_alu(int kind, uint32_t iters, uint32_t ctas_per_sm, uint32_t *dev_out, size_t out_words,
                                  void *cuda_stream, uint64_t *lane_ops)
{
    if (!dev_out || out_words < 1024 || ctas_per_sm < 1 || ctas_per_sm > 8) return VX_ERR_ARG;
    const unsigned grid = (unsigned)vx_sm_count() * ctas_per_sm;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    switch (kind) {
    case VX_PROBE_LOP3: vx_k_probe<VX_PROBE_LOP3><<<grid, VX_PROBE_THREADS, 0, st>>>(iters, 1u, dev_out); break;
    case VX_PROBE_SHF: vx_k_probe<VX_PROBE_SHF><<<grid, VX_PROBE_THREADS, 0, st>>>(iters, 1u, dev_out); break;
    case VX_PROBE_ADD: vx_k_probe<VX_PROBE_ADD><<<grid, VX_PROBE_THREADS, 0, st>>>(iters, 1u, dev_out); break;
    case VX_PROBE_IMAD: vx_k_probe<VX_PROBE_IMAD><<<grid, VX_PROBE_THREADS, 0, st>>>(iters, 1u, dev_out); break;
    case VX_PROBE_PRMT: vx_k_probe<VX_PROBE_PRMT><<<grid, VX_PROBE_THREADS, 0, st>>>(iters, 1u, dev_out); break;
    case VX_PROBE_ARX: vx_k_probe<VX_PROBE_ARX><<<grid, VX_PROBE_THREADS, 0, st>>>(iters, 1u, dev_out); break;
    default: return VX_ERR_ARG;
    }
    if (cudaGetLastError() != cudaSuccess) return VX_ERR_CUDA;
    if (lane_ops)
        *lane_ops = (uint64_t)grid * VX_PROBE_THREADS * (uint64_t)iters * VX_PROBE_UNROLL * VX_PROBE_CHAINS;
    return VX_OK;
}
