// vx_stage2.cu -- stage 2 of the plot: the fused sort + match kernel.
//
// PAPER.md L81 (III-A): "The sort and match stages are fused into a single GPU kernel, where each
// block is assigned one bucket, loads its nonces into shared memory, performs an insertion sort by
// hash value in shared memory, and then runs pairwise matching against an expected distance
// threshold to produce Table-2 records, with data never leaving shared memory between the two
// stages."  SURVEY.md 8(a) rows a6-a8.  The paper names its single-thread insertion sort as the
// O(n^2) bottleneck (L43, L123, L163) and a parallel sort as the fix (L165-169); this is that fix.
//
// One CTA owns one stage-1 partition at a time (a contiguous hash-prefix range holding 2^fb whole
// buckets, ~4096 records).  Hashes are uniform, so the sort is a distribution sort, O(n):
//   1. records -> registers; shared-memory atomics count them into 2^12 bins keyed by the next
//      12 hash bits below the partition prefix (about one record per bin);
//   2. exclusive scan of the bin counts; records scatter to bin start + claimed slot;
//   3. records of multi-record bins rank themselves inside the bin by (H, n)  -> fully sorted;
//   4. buckets are unions of bins (or sub-ranges of one bin at small K): CSR offsets fall out of
//      the scanned bin array;
//   5. match: each sorted record i scans forward while its successor is in the same bucket and
//      H_j - H_i < T = 2^(64-K)                                     (readings A11, A15);
//   6. Table-2 write positions need the number of matches of every earlier partition: a
//      decoupled look-back over partitions in ticket order supplies it in the same pass;
//   7. the sorted records leave shared memory once, as external-format Table 1 (reading A14), and
//      the matches as Table 2.
#include "vx_internal.h"

struct VxS2Params {
    const uint4 *part;           // stage-1 partition records {H lo, H hi, nonce lo, nonce hi}
    const uint32_t *cursor;
    const unsigned long long *part_base;
    unsigned long long *status;
    VxCtrl *ctrl;
    uint32_t *t1_rec;            // external Table-1 records as 32-bit words (3 per record)
    unsigned long long *t1_off;
    uint2 *t2_rec;               // external Table-2 records (nonce1, nonce2)
    unsigned long long *t2_off;
    unsigned long long N, NB, t2_cap;
    uint32_t P, cap, pb, fb, K, B, do_match;
};

#define VX_ST_AGG (1ull << 62)
#define VX_ST_INC (2ull << 62)
#define VX_ST_VAL ((1ull << 62) - 1)

__device__ __forceinline__ uint32_t vx_warp_incl_scan(uint32_t v, int lane)
{
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const uint32_t o = __shfl_up_sync(0xffffffffu, v, d);
        if (lane >= d) v += o;
    }
    return v;
}

// In-place exclusive scan of a[0..n) in shared memory, a[n] = total.  Conflict-free (each warp
// walks its own contiguous segment 32 words at a time).  All threads must call it.
template <int THREADS>
__device__ __forceinline__ void vx_block_exscan(uint32_t *a, int n, uint32_t *s_warp)
{
    constexpr int W = THREADS / 32;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int seg = ((n + W * 32 - 1) / (W * 32)) * 32;
    const int beg = min(warp * seg, n), end = min(beg + seg, n);
    uint32_t s = 0;
    for (int i = beg + lane; i < end; i += 32) s += a[i];
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) s += __shfl_xor_sync(0xffffffffu, s, d);
    if (lane == 0) s_warp[warp] = s;
    __syncthreads();
    const uint32_t w = lane < W ? s_warp[lane] : 0u;
    const uint32_t wi = vx_warp_incl_scan(w, lane);
    uint32_t carry = __shfl_sync(0xffffffffu, wi - w, warp);
    const uint32_t total = __shfl_sync(0xffffffffu, wi, W - 1);
    for (int i0 = beg; i0 < end; i0 += 32) {
        const int i = i0 + lane;
        const uint32_t v = i < end ? a[i] : 0u;
        const uint32_t incl = vx_warp_incl_scan(v, lane);
        if (i < end) a[i] = carry + incl - v;
        carry += __shfl_sync(0xffffffffu, incl, 31);
    }
    if (tid == 0) a[n] = total;
    __syncthreads();
}

// Decoupled look-back (warp 0 only, all 32 lanes): publishes this tile's aggregate, returns the
// sum of the aggregates of all tiles with a smaller ticket, then publishes the inclusive value.
__device__ __forceinline__ unsigned long long
vx_lookback(unsigned long long *status, uint32_t tile, unsigned long long aggregate, int lane)
{
    volatile unsigned long long *vs = status;
    if (tile == 0) {
        if (lane == 0) vs[0] = VX_ST_INC | aggregate;
        return 0;
    }
    if (lane == 0) vs[tile] = VX_ST_AGG | aggregate;
    unsigned long long excl = 0;
    long long j = (long long)tile - 1;
    for (;;) {
        const long long idx = j - lane;
        unsigned long long s = VX_ST_INC;   // lanes before tile 0 count as "inclusive, value 0"
        if (idx >= 0) {
            s = vs[idx];
            while ((s >> 62) == 0) { __nanosleep(20); s = vs[idx]; }
        }
        const unsigned incmask = __ballot_sync(0xffffffffu, (s >> 62) == 2);
        unsigned long long v = s & VX_ST_VAL;
        if (incmask) {
            const int first = __ffs(incmask) - 1;
            if (lane > first) v = 0;
        }
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) v += __shfl_xor_sync(0xffffffffu, v, d);
        excl += v;
        if (incmask) break;
        j -= 32;
    }
    if (lane == 0) vs[tile] = VX_ST_INC | (excl + aggregate);
    return excl;
}

template <int THREADS, int ITEMS>
__global__ void __launch_bounds__(THREADS, 2)
vx_k_sort_match(const __grid_constant__ VxS2Params q)
{
    extern __shared__ __align__(16) uint8_t vx_smem[];
    uint64_t *keyS = (uint64_t *)vx_smem;               // cap sorted hashes
    uint32_t *nonS = (uint32_t *)(keyS + q.cap);        // cap sorted nonces
    uint32_t *bins = nonS + q.cap;                      // VX_NBINS + 1 (+ pad)
    uint32_t *E = bins + VX_NBINS + 32;                 // cap + 1 match-count prefix
    __shared__ uint32_t s_warp[32];
    __shared__ uint32_t s_tile;
    __shared__ unsigned long long s_base2;

    const int tid = threadIdx.x, lane = tid & 31;
    const int binshift = 64 - (int)q.pb - VX_BIN_BITS;
    const int bshift = 64 - (int)q.B;                   // bucket = H >> bshift
    const uint32_t fbmask = (1u << q.fb) - 1u;
    const unsigned long long T = 1ull << (64 - q.K);
    uint32_t cta_max_bucket = 0;

    for (;;) {
        __syncthreads();                                // previous tile fully drained
        if (tid == 0) s_tile = atomicAdd(&q.ctrl->ticket, 1u);
        for (int i = tid; i <= (int)VX_NBINS; i += THREADS) bins[i] = 0;
        __syncthreads();
        const uint32_t tile = s_tile;
        if (tile >= q.P) break;

        const uint32_t cnt = min(q.cursor[tile], q.cap);
        const unsigned long long base1 = q.part_base[tile];
        const uint4 *src = q.part + (size_t)tile * q.cap;

        // ---- 1. load + bin count -------------------------------------------------------------
        uint64_t key[ITEMS];
        uint32_t non[ITEMS], slot[ITEMS];
#pragma unroll
        for (int it = 0; it < ITEMS; it++) {
            const uint32_t idx = it * THREADS + tid;
            const uint4 r = idx < cnt ? __ldg(src + idx) : make_uint4(0u, 0u, 0u, 0u);
            key[it] = ((uint64_t)r.y << 32) | r.x;
            non[it] = r.z;
        }
#pragma unroll
        for (int it = 0; it < ITEMS; it++) {
            const uint32_t idx = it * THREADS + tid;
            if (idx < cnt) slot[it] = atomicAdd(&bins[(uint32_t)(key[it] >> binshift) & (VX_NBINS - 1)], 1u);
        }
        __syncthreads();
        // ---- 2. scan + scatter ---------------------------------------------------------------
        vx_block_exscan<THREADS>(bins, (int)VX_NBINS, s_warp);
#pragma unroll
        for (int it = 0; it < ITEMS; it++) {
            const uint32_t idx = it * THREADS + tid;
            if (idx < cnt) {
                const uint32_t pos = bins[(uint32_t)(key[it] >> binshift) & (VX_NBINS - 1)] + slot[it];
                keyS[pos] = key[it];
                nonS[pos] = non[it];
            }
        }
        __syncthreads();
        // ---- 3. rank inside multi-record bins ------------------------------------------------
#pragma unroll
        for (int it = 0; it < ITEMS; it++) {
            const uint32_t idx = it * THREADS + tid;
            slot[it] = 0xffffffffu;                     // "stays where it is"
            if (idx < cnt) {
                const uint32_t b = (uint32_t)(key[it] >> binshift) & (VX_NBINS - 1);
                const uint32_t s = bins[b], e = bins[b + 1];
                if (e - s > 1) {
                    uint32_t rank = 0;
                    for (uint32_t j = s; j < e; j++) {
                        const uint64_t kj = keyS[j];
                        rank += (kj < key[it] || (kj == key[it] && nonS[j] < non[it])) ? 1u : 0u;
                    }
                    slot[it] = s + rank;
                }
            }
        }
        __syncthreads();
#pragma unroll
        for (int it = 0; it < ITEMS; it++)
            if (slot[it] != 0xffffffffu) { keyS[slot[it]] = key[it]; nonS[slot[it]] = non[it]; }
        __syncthreads();

        // first sorted position of local bucket bl (bl == 2^fb gives cnt)
        auto bucket_start = [&](uint32_t bl) -> uint32_t {
            if (q.fb <= VX_BIN_BITS) return bins[bl << (VX_BIN_BITS - q.fb)];
            const uint32_t b = bl >> (q.fb - VX_BIN_BITS);
            if (b >= VX_NBINS) return cnt;
            uint32_t s = bins[b];
            const uint32_t e = bins[b + 1];
            while (s < e && ((uint32_t)(keyS[s] >> bshift) & fbmask) < bl) s++;
            return s;
        };

        // ---- 5. match count ------------------------------------------------------------------
        unsigned long long base2 = 0;
        uint32_t M = 0;
        if (q.do_match) {
            for (uint32_t i = tid; i < cnt; i += THREADS) {
                const uint64_t ki = keyS[i];
                uint32_t c = 0;
                for (uint32_t j = i + 1; j < cnt; j++) {
                    const uint64_t kj = keyS[j];
                    if (((kj ^ ki) >> bshift) != 0 || kj - ki >= T) break;
                    c++;
                }
                E[i] = c;
            }
            __syncthreads();
            vx_block_exscan<THREADS>(E, (int)cnt, s_warp);
            M = E[cnt];
            // ---- 6. look-back for the Table-2 base ---------------------------------------------
            if (tid < 32) {
                const unsigned long long b2 = vx_lookback(q.status, tile, M, lane);
                if (tid == 0) s_base2 = b2;
            }
            __syncthreads();
            base2 = s_base2;
            if (base2 + M > q.t2_cap) {
                if (tid == 0) atomicOr(&q.ctrl->flags, VX_FLAG_T2_OVERFLOW);
            } else {
                for (uint32_t i = tid; i < cnt; i += THREADS) {
                    const uint64_t ki = keyS[i];
                    const uint32_t ni = nonS[i];
                    uint2 *dst = q.t2_rec + (base2 + E[i]);
                    for (uint32_t j = i + 1; j < cnt; j++) {
                        const uint64_t kj = keyS[j];
                        if (((kj ^ ki) >> bshift) != 0 || kj - ki >= T) break;
                        *dst++ = make_uint2(ni, nonS[j]);
                    }
                }
            }
        }
        // ---- 4. CSR offsets of this partition's buckets ----------------------------------------
        {
            const uint32_t nb_local = 1u << q.fb;
            const unsigned long long gb0 = (unsigned long long)tile << q.fb;
            for (uint32_t bl = tid; bl < nb_local; bl += THREADS) {
                const uint32_t s = bucket_start(bl), e = bucket_start(bl + 1);
                cta_max_bucket = max(cta_max_bucket, e - s);
                q.t1_off[gb0 + bl] = base1 + s;
                if (q.do_match) q.t2_off[gb0 + bl] = base2 + E[s];
            }
            if (tile == q.P - 1 && tid == 0) {
                q.t1_off[q.NB] = base1 + cnt;
                if (q.do_match) {
                    q.t2_off[q.NB] = base2 + M;
                    q.ctrl->t2_total = base2 + M;
                }
            }
        }
        // ---- 7. sorted Table 1, external format: nonce LE | digest bytes 0..7 -------------------
        {
            uint32_t *dst = q.t1_rec + base1 * 3ull;
            const uint32_t words = cnt * 3u;
            for (uint32_t w = tid; w < words; w += THREADS) {
                const uint32_t r = w / 3u, f = w - 3u * r;
                uint32_t val;
                if (f == 0) val = nonS[r];
                else {
                    const uint64_t k = keyS[r];
                    val = __byte_perm(f == 1 ? (uint32_t)(k >> 32) : (uint32_t)k, 0, 0x0123);
                }
                dst[w] = val;
            }
        }
    }
    // largest bucket, one atomic per CTA
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) cta_max_bucket = max(cta_max_bucket, __shfl_xor_sync(0xffffffffu, cta_max_bucket, d));
    if (lane == 0 && cta_max_bucket) atomicMax(&q.ctrl->max_bucket, cta_max_bucket);
}

size_t vx_stage2_smem_bytes(const VxGeom &g)
{
    return (size_t)g.cap * 8 + (size_t)g.cap * 4 + (VX_NBINS + 32) * 4 + ((size_t)g.cap + 32) * 4;
}

cudaError_t vx_stage2_configure(void)
{
    return cudaFuncSetAttribute(vx_k_sort_match<VX_S2_THREADS, VX_S2_ITEMS>,
                                cudaFuncAttributeMaxDynamicSharedMemorySize, 110 * 1024);
}

cudaError_t vx_launch_stage2(const VxGeom &g, uint8_t *ws, bool do_match, int num_sms, cudaStream_t st)
{
    VxCtrl *ctrl = (VxCtrl *)(ws + g.off_ctrl);
    cudaError_t e = cudaMemsetAsync(&ctrl->ticket, 0, sizeof(uint32_t), st);
    if (e != cudaSuccess) return e;
    e = cudaMemsetAsync(&ctrl->max_bucket, 0, sizeof(uint32_t), st);
    if (e != cudaSuccess) return e;
    e = cudaMemsetAsync(ws + g.off_status, 0, g.P * sizeof(unsigned long long), st);
    if (e != cudaSuccess) return e;
    VxS2Params q;
    q.part = (const uint4 *)(ws + g.off_part);
    q.cursor = (const uint32_t *)(ws + g.off_cursor);
    q.part_base = (const unsigned long long *)(ws + g.off_part_base);
    q.status = (unsigned long long *)(ws + g.off_status);
    q.ctrl = ctrl;
    q.t1_rec = (uint32_t *)(ws + g.off_t1_rec);
    q.t1_off = (unsigned long long *)(ws + g.off_t1_off);
    q.t2_rec = (uint2 *)(ws + g.off_t2_rec);
    q.t2_off = (unsigned long long *)(ws + g.off_t2_off);
    q.N = g.N; q.NB = g.NB; q.t2_cap = g.t2_cap;
    q.P = (uint32_t)g.P; q.cap = g.cap; q.pb = g.pb; q.fb = g.fb; q.K = g.K; q.B = g.B;
    q.do_match = do_match ? 1u : 0u;
    const size_t smem = vx_stage2_smem_bytes(g);
    uint64_t grid = (uint64_t)num_sms * 2;
    if (grid > g.P) grid = g.P;
    vx_k_sort_match<VX_S2_THREADS, VX_S2_ITEMS><<<(unsigned)grid, VX_S2_THREADS, smem, st>>>(q);
    return cudaGetLastError();
}
