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
//   A. records -> registers; shared-memory atomics count them into 2^12 bins keyed by the next
//      12 hash bits below the partition prefix (about one record per bin) and hand out slots;
//   B. exclusive scan of the bin counts, 8 bins per thread in registers;
//   C. records scatter to bin start + slot;
//   D. records of multi-record bins rank themselves inside the bin by H -> fully sorted.  Equal
//      64-bit hashes (about 2^(2K-65) pairs per plot) raise a flag and the tile re-ranks by (H, n);
//   E. match count, one lane per sorted position: c_i = number of successors j with
//      H_j <= min(H_i + T - 1, last hash of the bucket), T = 2^(64-K)     (readings A11, A15);
//      the matches of i are exactly the records i+1 .. i+c_i;
//   F. exclusive scan of c_i; the tile's total is published for the decoupled look-back that
//      supplies the Table-2 base of the tile (ticket order = partition order);
//   G. the sorted partition goes back to HBM IN PLACE (reading A14) -- Table 1 stays resident as
//      sorted buckets inside the partition array, 16-byte records -- and the bucket offsets
//      (CSR) are written, while the look-back resolves;
//   H. Table-2 records (n_i, n_j) are written at base + E_i + t.
#include "vx_internal.h"

struct VxS2Params {
    uint4 *part;                 // partition records {H lo, H hi, nonce lo, nonce hi}; sorted in place
                                 // (wide: uint64 a = (H << pb) | (n >> 12), with part_b: uint16 n & 0xfff)
    uint16_t *part_b;
    uint8_t *t2_hi;              // wide: (n1 >> 32) | (n2 >> 32) << 4 per Table-2 record
    // sort key geometry (host-computed; the sort key is H, or a in the wide layout):
    unsigned long long Tm1;      // (T - 1) in key units: (2^(64-K) - 1) << (wide ? pb : 0)
    unsigned long long bmask;    // key | bmask = largest key of the key's bucket
    unsigned long long lowmask;  // wide: the low pb key bits that hold nonce bits, else 0
    uint32_t nlo_bits;           // wide: nonce bits kept in part_b (= tile_log)
    int binshift, bshift;        // bin = (key >> binshift) & (NBINS-1); bucket-in-tile = (key >> bshift) & fbmask
    const uint32_t *cursor;
    const unsigned long long *part_base;
    unsigned long long *status;
    VxCtrl *ctrl;
    unsigned long long *t1_off;
    uint2 *t2_rec;               // external Table-2 records (nonce1, nonce2)
    unsigned long long *t2_off;
    unsigned long long N, NB, t2_cap;   // NB: buckets of this pass (all 2^B unless the plot is made in passes)
    uint32_t P, cap, pb, fb, K, B, do_match, force_exact;
    uint32_t submask;            // sub-key bits the fast ranking pass compares (~0; a test hook narrows it)
    // this launch sorts the partitions [tile_begin, tile_end): the whole plot, or one slice of it
    // when Table 2 is streamed to the host while later slices are still being matched (vx_egress.cu)
    uint32_t tile_begin, tile_end;
    uint32_t cap_check;          // records a partition may hold (= cap unless a test lowered it)
    unsigned long long *slice_end_out;   // host-mapped: |Table 2| after partition tile_end - 1, or NULL
};

#define VX_ST_AGG (1ull << 62)
#define VX_ST_INC (2ull << 62)
#define VX_ST_VAL ((1ull << 62) - 1)
#define VX_FULL 0xffffffffu

#ifndef VX_EXP_TMA
#define VX_EXP_TMA 0
#endif
#if VX_EXP_TMA
// experiment (DESIGN.md 6.2 "TMA staging"): the partition comes into shared memory by cp.async.bulk with an
// mbarrier, in two halves through the (then free) sorted-key array, instead of by per-thread global loads
__device__ __forceinline__ uint32_t vx_smem_addr(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void vx_mbar_init(void *bar) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" :: "r"(vx_smem_addr(bar)) : "memory");
}
__device__ __forceinline__ void vx_tma_load(void *dst, const void *src, uint32_t bytes, void *bar) {
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" :: "r"(vx_smem_addr(bar)), "r"(bytes) : "memory");
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 :: "r"(vx_smem_addr(dst)), "l"(src), "r"(bytes), "r"(vx_smem_addr(bar)) : "memory");
}
__device__ __forceinline__ void vx_mbar_wait(void *bar, uint32_t parity) {
    asm volatile("{\n.reg .pred p;\nVX_WAIT:\nmbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n@p bra VX_DONE;\nbra VX_WAIT;\nVX_DONE:\n}"
                 :: "r"(vx_smem_addr(bar)), "r"(parity) : "memory");
}
#endif

__device__ __forceinline__ uint32_t vx_warp_incl_scan(uint32_t v, int lane)
{
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const uint32_t o = __shfl_up_sync(VX_FULL, v, d);
        if (lane >= d) v += o;
    }
    return v;
}

// In-place exclusive scan of a[0 .. THREADS*IPT) in shared memory; thread t owns the IPT
// consecutive entries starting at t*IPT and scans them in registers.  Returns the total to every
// thread.  The caller synchronises before anybody reads a[] again.  All threads must call it.
template <int THREADS, int IPT>
__device__ __forceinline__ uint32_t vx_block_exscan(uint32_t *a, uint32_t *s_warp)
{
    constexpr int W = THREADS / 32;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    uint32_t v[IPT];
    if constexpr (IPT % 4 == 0) {
#pragma unroll
        for (int k = 0; k < IPT / 4; k++) {
            const uint4 q = reinterpret_cast<const uint4 *>(a)[tid * (IPT / 4) + k];
            v[4 * k] = q.x; v[4 * k + 1] = q.y; v[4 * k + 2] = q.z; v[4 * k + 3] = q.w;
        }
    } else {
#pragma unroll
        for (int k = 0; k < IPT; k++) v[k] = a[tid * IPT + k];
    }
    uint32_t sum = 0;
#pragma unroll
    for (int k = 0; k < IPT; k++) { const uint32_t t = v[k]; v[k] = sum; sum += t; }
    const uint32_t incl = vx_warp_incl_scan(sum, lane);
    if (lane == 31) s_warp[warp] = incl;
    __syncthreads();
    const uint32_t w = lane < W ? s_warp[lane] : 0u;
    const uint32_t total = __reduce_add_sync(VX_FULL, w);
    const uint32_t base = __reduce_add_sync(VX_FULL, lane < warp ? w : 0u) + incl - sum;
    if constexpr (IPT % 4 == 0) {
#pragma unroll
        for (int k = 0; k < IPT / 4; k++)
            reinterpret_cast<uint4 *>(a)[tid * (IPT / 4) + k] =
                make_uint4(v[4 * k] + base, v[4 * k + 1] + base, v[4 * k + 2] + base, v[4 * k + 3] + base);
    } else {
#pragma unroll
        for (int k = 0; k < IPT; k++) a[tid * IPT + k] = v[k] + base;
    }
    return total;
}

// Decoupled look-back (warp 0 only, all 32 lanes).  The tile's aggregate has already been
// published (VX_ST_AGG); returns the sum of the aggregates of all tiles with a smaller ticket and
// publishes the inclusive value.
__device__ __forceinline__ unsigned long long
vx_lookback(unsigned long long *status, uint32_t tile, unsigned long long aggregate, int lane)
{
    volatile unsigned long long *vs = status;
    if (tile == 0) {
        if (lane == 0) vs[0] = VX_ST_INC | aggregate;
        return 0;
    }
    unsigned long long excl = 0;
    long long j = (long long)tile - 1;
    for (;;) {
        const long long idx = j - lane;
        unsigned long long s = VX_ST_INC;   // lanes before tile 0 count as "inclusive, value 0"
        if (idx >= 0) {
            s = vs[idx];
            for (unsigned ns = 128; (s >> 62) == 0; ns = min(ns * 2u, 1024u)) { __nanosleep(ns); s = vs[idx]; }
        }
        const unsigned incmask = __ballot_sync(VX_FULL, (s >> 62) == 2);
        unsigned long long v = s & VX_ST_VAL;
        if (incmask) {
            const int first = __ffs(incmask) - 1;
            if (lane > first) v = 0;
        }
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) v += __shfl_xor_sync(VX_FULL, v, d);
        excl += v;
        if (incmask) break;
        j -= 32;
    }
    if (lane == 0) vs[tile] = VX_ST_INC | (excl + aggregate);
    return excl;
}

// the 32 hash bits right below the bin index (bin = (H >> binshift) & (VX_NBINS - 1)); the caller masks
// off the low 4 (the record's slot in its bin goes there) and whatever a test hook narrows.  binshift >= 32
// always (pb + VX_BIN_BITS <= 32; checked at launch), so both are 32-bit operations on the high word:
// sh = binshift - 32
__device__ __forceinline__ uint32_t vx_subkey(uint64_t k, int sh)
{
    return __funnelshift_r((uint32_t)k, (uint32_t)(k >> 32), sh);
}
template <uint32_t NBINS>
__device__ __forceinline__ uint32_t vx_bin(uint64_t k, int sh)
{
    return ((uint32_t)(k >> 32) >> sh) & (NBINS - 1);
}

// Two tile geometries are built (vx_internal.h): 2^12-record tiles, 512 threads, 2 CTAs per SM
// (K <= 31) and 2^13-record tiles, 1024 threads, 1 CTA per SM (K >= 32, where stage 1 cannot keep
// 2^(K-12) open partitions resident in L2).  BIN_BITS = log2 of the tile size: one bin per record.
template <int THREADS, int ITEMS, int BIN_BITS, int MINB, bool WIDE>
__global__ void __launch_bounds__(THREADS, MINB)
vx_k_sort_match(const __grid_constant__ VxS2Params q)
{
    constexpr uint32_t VX_NBINS = 1u << BIN_BITS;       // (shadows nothing: the macros are gone)
    constexpr int VX_BIN_BITS = BIN_BITS;
    constexpr int CAPA = THREADS * ITEMS;               // allocated sorted positions
    extern __shared__ __align__(16) uint8_t vx_smem[];
    uint64_t *keyS = (uint64_t *)vx_smem;               // CAPA sorted hashes + sentinel (+ pad)
    uint32_t *nonS = (uint32_t *)(keyS + CAPA + 8);     // CAPA sorted nonces (low 32 bits)
    uint32_t *bins = nonS + CAPA;                       // VX_NBINS + 1 (+ pad)
    uint32_t *E = bins + VX_NBINS + 32;                 // CAPA + 1 (+ pad): match-count prefix
    uint32_t *sub = E;                                  // phases C-D only: 32-bit ranking sub-keys
    // wide layout: bits 32.. of every sorted record's nonce, one byte each (+ pad), filled by phase G for the
    // emit (which then finds the low 32 nonce bits in nonS, like the narrow one)
    uint8_t *hiS = (uint8_t *)(E + CAPA + 32);
    __shared__ uint32_t s_warp[32];
    __shared__ uint32_t s_tile, s_tie, s_cnt;
#if VX_EXP_TMA
    __shared__ __align__(8) unsigned long long s_mbar;
    uint32_t par = 0;                                   // phase parity of s_mbar, the same in every thread
    constexpr uint32_t VX_HALF = CAPA / 2;              // records per staging chunk: the sorted-key array holds half a tile
    if (threadIdx.x == 0) vx_mbar_init(&s_mbar);        // (the barrier at the top of the tile loop publishes it)
#endif
    __shared__ unsigned long long s_base2;
    // deferred emit (phase H of tile t runs after phase A of the CTA's next tile): Table-2 prefix at
    // the first record of every bucket of tile t, saved before the bins are recycled
    constexpr uint32_t VX_DEFER_MAXB = 512;
    __shared__ uint32_t s_e2[VX_DEFER_MAXB];

    const int tid = threadIdx.x, lane = tid & 31, wbase = tid & ~31;
    const int sh = q.binshift - 32;                     // bin / sub-key shifts act on the high key word
    const uint32_t submask = q.submask;
    const int bshift = q.bshift;
    const uint32_t fbmask = (1u << q.fb) - 1u;
    const uint64_t Tm1 = q.Tm1;                         // T - 1 in key units
    const uint64_t bmask = q.bmask;                     // key | bmask = last key of the key's bucket
    uint32_t cta_max_bucket = 0;
    const uint32_t nb_local = 1u << q.fb;
    // The Table-2 base of a tile comes from the decoupled look-back over all earlier tiles, and the
    // ~300 tiles in flight run a few microseconds apart: emitting right after the write-back left
    // the CTA waiting 13 % of its time.  So a tile's look-back + emit (phase H) are deferred until
    // the CTA has loaded and binned its NEXT tile (phase A touches only registers and the bins):
    // the predecessors get that much longer to publish their totals.
    const bool defer = q.do_match && nb_local <= VX_DEFER_MAXB;
    bool pending = false;                               // CTA-uniform
    // (tile, count and matches of the tile whose emit is pending: CTA-uniform, so they live in shared
    // memory rather than in three registers of every thread -- the kernel sits at its register limit)
    __shared__ uint32_t s_p[3];

    // ---- look-back for the Table-2 base, then H: the matches of i are i+1 .. i+c_i, c_i = E[i+1] - E[i]
    auto lookback_emit = [&](uint32_t tile, uint32_t cnt, uint32_t M) {
        if (tid < 32) {
#ifdef VX_EXP_NO_LOOKBACK
            // measurement only: no look-back, Table 2 lands at tile * 4000 -- WRONG tables, right timing
            const unsigned long long b2 = (unsigned long long)tile * 4000ull;
#else
            const unsigned long long b2 = vx_lookback(q.status, tile, M, lane);
#endif
            if (tid == 0) {
                s_base2 = b2;
                if (tile == q.tile_end - 1 && q.slice_end_out) *q.slice_end_out = b2 + M;
            }
        }
        __syncthreads();
        const unsigned long long base2 = s_base2;
        if (base2 + M > q.t2_cap) {
            if (tid == 0) atomicOr(&q.ctrl->flags, VX_FLAG_T2_OVERFLOW);
        } else {
#pragma unroll
            for (int it = 0; it < ITEMS; it++) {
                if (it * THREADS + wbase < cnt) {
                    const uint32_t i = it * THREADS + tid;
                    const uint32_t e0 = E[i];
                    const uint32_t c = E[i + 1] - e0;
                    VX_CHECK(q.ctrl, i + 1 <= (uint32_t)CAPA && e0 + c <= M && (c == 0 || i + c < cnt) && base2 + e0 + c <= q.t2_cap);
                    const uint32_t cmax = __reduce_max_sync(VX_FULL, c);
                    if (cmax) {
                        if constexpr (WIDE) {
                            // phase G left the low 32 bits of every sorted record's nonce in nonS and the bits above
                            // them in hiS: the emit is the narrow one plus a byte of high bits per Table-2 record.
                            // The first four successors unconditionally (positions up to CAPA + 3 lie inside the
                            // arrays' padding), their loads issued together ahead of the stores; longer runs take the loop
                            const uint32_t ni = nonS[i], nih = hiS[i];
                            const uint32_t *np = nonS + i + 1;
                            const uint8_t *hp = hiS + i + 1;
                            uint2 *dst = q.t2_rec + (base2 + e0);
                            uint8_t *dsth = q.t2_hi + (base2 + e0);
                            // (both pointers pinned in registers: ptxas otherwise rebuilds the byte pointer from the
                            // index for every store, behind a branch of its own -- 7 instructions per byte)
                            asm volatile("" : "+l"(dst), "+l"(dsth));
                            __builtin_assume(__isGlobal(dst));
                            __builtin_assume(__isGlobal(dsth));
                            uint32_t nj[4], hj[4];
#pragma unroll
                            for (uint32_t t = 0; t < 4; t++) { nj[t] = np[t]; hj[t] = hp[t]; }
#pragma unroll
                            for (uint32_t t = 0; t < 4; t++) hj[t] = nih | (hj[t] << 4);
#pragma unroll
                            for (uint32_t t = 0; t < 4; t++)
                                if (t < c) {
                                    dst[t] = make_uint2(ni, nj[t]);
                                    dsth[t] = (uint8_t)hj[t];
                                }
                            for (uint32_t t = 4; t < cmax; t++)
                                if (t < c) {
                                    dst[t] = make_uint2(ni, np[t]);
                                    dsth[t] = (uint8_t)(nih | ((uint32_t)hp[t] << 4));
                                }
                        } else {
                            const uint32_t ni = nonS[i];
                            const uint32_t *np = nonS + i + 1;
                            uint2 *dst = q.t2_rec + (base2 + e0);
                            // (pinned in registers: ptxas otherwise rebuilds the pointer from the index for every store)
                            asm volatile("" : "+l"(dst));
                            __builtin_assume(__isGlobal(dst));
#pragma unroll
                            for (uint32_t t = 0; t < 4; t++)
                                if (t < c) dst[t] = make_uint2(ni, np[t]);
                            for (uint32_t t = 4; t < cmax; t++)
                                if (t < c) dst[t] = make_uint2(ni, np[t]);
                        }
                    }
                }
            }
        }
        return base2;
    };

    for (;;) {
        __syncthreads();                                // previous tile fully drained
        if (tid == 0) {
            const uint32_t t = q.tile_begin + atomicAdd(&q.ctrl->ticket, 1u);
            s_tile = t;
            // the tile's record count travels with the ticket: one thread's load behind the atomic instead of
            // every thread's load behind the barrier
            s_cnt = t < q.tile_end ? min(q.cursor[t], q.cap_check) : 0u;
            // Tickets are handed out in partition order and the CTAs run about one tile apart, so the
            // partition gridDim tickets ahead is the one some CTA (most likely this one) takes next:
            // one bulk prefetch (TMA, cp.async.bulk.prefetch.L2 -> UBLKPF.L2) brings its 64 KB into
            // L2 while this tile is sorted, and phase A's loads no longer wait for HBM (K=31:
            // 33.9 -> 32.7 ms).  A hint only: nothing depends on who takes that partition, or when.
            const uint32_t pf = t + gridDim.x;
            if (pf < q.tile_end) {
                const uint32_t n = min(q.cursor[pf], q.cap_check);
                const char *p = reinterpret_cast<const char *>(q.part) + (size_t)pf * q.cap * (WIDE ? 8 : 16);
                const uint32_t bytes = n * (WIDE ? 8u : 16u) & ~15u;
                if (bytes) asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" :: "l"(p), "r"(bytes) : "memory");
                if constexpr (WIDE) {
                    const char *pb2 = reinterpret_cast<const char *>(q.part_b) + (size_t)pf * q.cap * 2;
                    const uint32_t b2 = n * 2u & ~15u;
                    if (b2) asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" :: "l"(pb2), "r"(b2) : "memory");
                }
            }
        }
        // exact = rank by (H, n) with full compares; the fast pass ranks by H alone and is
        // validated in phase E (a tile holding two equal hashes comes back for an exact pass)
        uint32_t exact = q.force_exact | (q.do_match ^ 1u);
        uint32_t tile, cnt;
        uint4 *src;
        unsigned short *src_b = nullptr;
        uint64_t key[ITEMS];
        uint32_t non[ITEMS], sn[ITEMS];                 // sn: slot, later position | bin size << 16
        uint32_t M = 0;
        bool finished = false;
        for (;;) {
#if VX_EXP_TMA
            if constexpr (!WIDE) {
                if (tid == 0 && s_cnt)                  // first half of the partition -> the sorted-key array (free here)
                    vx_tma_load(keyS, q.part + (size_t)s_tile * q.cap, min(s_cnt, VX_HALF) * 16u, &s_mbar);
            }
#endif
            for (int i = tid; i < (int)(VX_NBINS + 32) / 4; i += THREADS)
                reinterpret_cast<uint4 *>(bins)[i] = make_uint4(0u, 0u, 0u, 0u);
            __syncthreads();
            if (tid == 0) s_tie = 0u;                   // set in phase E, read after the sync behind it
            tile = s_tile;
            const bool valid = tile < q.tile_end;
            cnt = s_cnt;
            if constexpr (WIDE) {
                src = reinterpret_cast<uint4 *>(reinterpret_cast<unsigned long long *>(q.part) + (size_t)tile * q.cap);
                src_b = q.part_b + (size_t)tile * q.cap;
            } else {
                src = q.part + (size_t)tile * q.cap;
            }

            // ---- A. load + bin count -----------------------------------------------------------
#if VX_EXP_TMA
            if constexpr (!WIDE) {
                const uint4 *stage = reinterpret_cast<const uint4 *>(keyS);
                if (cnt) { vx_mbar_wait(&s_mbar, par); par ^= 1u; }
#pragma unroll
                for (int it = 0; it < ITEMS; it++) {
                    const uint32_t idx = it * THREADS + tid;
                    key[it] = 0ull; non[it] = 0u;
                    if (idx < cnt && idx < VX_HALF) {
                        const uint4 r = stage[idx];
                        key[it] = ((uint64_t)r.y << 32) | r.x;
                        non[it] = r.z;
                    }
                }
                if (cnt > VX_HALF) {                    // CTA-uniform
                    __syncthreads();                    // everybody has taken its records of the first half
                    if (tid == 0) vx_tma_load(keyS, src + VX_HALF, (cnt - VX_HALF) * 16u, &s_mbar);
                    vx_mbar_wait(&s_mbar, par); par ^= 1u;
#pragma unroll
                    for (int it = 0; it < ITEMS; it++) {
                        const uint32_t idx = it * THREADS + tid;
                        if (idx < cnt && idx >= VX_HALF) {
                            const uint4 r = stage[idx - VX_HALF];
                            key[it] = ((uint64_t)r.y << 32) | r.x;
                            non[it] = r.z;
                        }
                    }
                }
                __syncthreads();                        // staging read; phase C may write the sorted keys
            } else
#endif
            {
#pragma unroll
            for (int it = 0; it < ITEMS; it++) {
                const uint32_t idx = it * THREADS + tid;
                if constexpr (WIDE) {
                    key[it] = idx < cnt ? __ldcs(reinterpret_cast<const unsigned long long *>(src) + idx) : 0ull;
                    non[it] = idx < cnt ? __ldcs(src_b + idx) : 0u;
                } else {
                    const uint4 r = idx < cnt ? __ldcs(src + idx) : make_uint4(0u, 0u, 0u, 0u);
                    key[it] = ((uint64_t)r.y << 32) | r.x;
                    non[it] = r.z;
                }
            }
            }
#pragma unroll
            for (int it = 0; it < ITEMS; it++) {
                const uint32_t idx = it * THREADS + tid;
                VX_CHECK(q.ctrl, cnt <= (uint32_t)CAPA && cnt <= q.cap && vx_bin<VX_NBINS>(key[it], sh) < VX_NBINS);
                if (idx < cnt) sn[it] = atomicAdd(&bins[vx_bin<VX_NBINS>(key[it], sh)], 1u);
            }
            if (pending) {                              // the previous tile of this CTA: look-back + H
                const uint32_t p_tile = s_p[0], p_M = s_p[2];
                const unsigned long long base2 = lookback_emit(p_tile, s_p[1], p_M);
                const unsigned long long pg0 = (unsigned long long)p_tile << q.fb;
                for (uint32_t bl = tid; bl < nb_local; bl += THREADS) q.t2_off[pg0 + bl] = base2 + s_e2[bl];
                if (p_tile == q.P - 1 && tid == 0) {
                    q.t2_off[q.NB] = base2 + p_M;
                    q.ctrl->t2_total = base2 + p_M;
                }
                pending = false;
            }
            if (!valid) { finished = true; break; }
            __syncthreads();
            // ---- B. scan -------------------------------------------------------------------------
            {
                const uint32_t total = vx_block_exscan<THREADS, VX_NBINS / THREADS>(bins, s_warp);
                if (tid == 0) bins[VX_NBINS] = total;
            }
            __syncthreads();
            // ---- C. scatter to bin start + slot (bank-random, the only such pass) ------------------
            // sub[] = the 32 hash bits below the bin index: what the fast ranking pass compares
            //      (all bin starts are fetched before the first store: nine independent loads in flight)
            {
                uint32_t pos[ITEMS];
#pragma unroll
                for (int it = 0; it < ITEMS; it++) {
                    const uint32_t idx = it * THREADS + tid;
                    pos[it] = idx < cnt ? bins[vx_bin<VX_NBINS>(key[it], sh)] + sn[it] : 0xffffffffu;
                }
#pragma unroll
                for (int it = 0; it < ITEMS; it++) {
                    if (pos[it] != 0xffffffffu) {
                        VX_CHECK(q.ctrl, pos[it] < cnt);
                        keyS[pos[it]] = key[it];
                        nonS[pos[it]] = non[it];
                        // ranking key: the hash bits below the bin index with the record's slot in the bin
                        // (its arrival order, unique there) in the low 4 bits -- distinct within a bin, so the
                        // ranks below are distinct and no two lanes ever write one sorted slot
                        sub[pos[it]] = (vx_subkey(key[it], sh) & submask) | sn[it];
                        if (sn[it] > 15u) s_tie = 1u;   // a bin of more than 16 records: rank it exactly
                    }
                }
            }
            if (tid < 8) keyS[cnt + tid] = ~0ull;       // sentinels behind the last record: no clamps in E
            __syncthreads();
            // ---- D. rank inside multi-record bins, one lane per position (neighbouring lanes
            //         read neighbouring bins: conflict-free), warp lock-step over the largest bin -----
#pragma unroll
            for (int it = 0; it < ITEMS; it++) {
                if (it * THREADS + wbase < cnt) {
                    const uint32_t i = it * THREADS + tid;
                    const uint64_t k = keyS[i];         // i >= cnt: sentinel or stale, result unused
                    const uint32_t nn = nonS[i];
                    const uint32_t b = vx_bin<VX_NBINS>(k, sh);
                    const uint32_t s = bins[b];
                    uint32_t n = bins[b + 1] - s;
                    VX_CHECK(q.ctrl, b < VX_NBINS && (i >= cnt || (s <= i && i < s + n && s + n <= cnt)));
                    if (i >= cnt || n == 1) n = 0;      // alone in its bin: stays
                    const uint32_t nm = __reduce_max_sync(VX_FULL, n);
                    uint32_t rank = 0;
                    if (!exact) {
                        // by the ranking key of phase C: (27 hash bits below the bin index, slot in the bin).
                        // Every record of a bin gets a rank of its own.  Records that tie on those hash bits
                        // may come out in the wrong order, which phase E sees as keys that do not strictly
                        // increase (about 8 tiles of a K = 31 plot), as it does two equal hashes
                        const uint32_t *sp = sub + s;
                        const uint32_t ks = sub[i];
#pragma unroll
                        for (uint32_t j = 0; j < 4; j++) {
                            const uint32_t kj = j < n ? sp[j] : 0xffffffffu;
                            rank += kj < ks ? 1u : 0u;
                        }
                        if (nm > 4) {
#pragma unroll 1
                            for (uint32_t j = 4; j < nm; j++) {
                                const uint32_t kj = j < n ? sp[j] : 0xffffffffu;
                                rank += kj < ks ? 1u : 0u;
                            }
                        }
                    } else {                            // by (H, n), reading A10
                        const uint64_t *kp = keyS + s;
                        const uint32_t *np = nonS + s;
#pragma unroll 1
                        for (uint32_t j = 0; j < nm; j++)
                            if (j < n) rank += (kp[j] < k || (kp[j] == k && np[j] < nn)) ? 1u : 0u;
                    }
                    key[it] = k;
                    non[it] = nn;
                    sn[it] = (s + rank) | (n << 16);
                }
            }
            __syncthreads();
#pragma unroll
            for (int it = 0; it < ITEMS; it++) {
                if (it * THREADS + wbase < cnt) {
                    if (sn[it] >> 16) {
                        const uint32_t pos = sn[it] & 0xffffu;
                        VX_CHECK(q.ctrl, pos < cnt);
                        keyS[pos] = key[it];
                        nonS[pos] = non[it];
                    }
                }
            }
            __syncthreads();
            // ---- E. match count: lane i counts its successors within reach ----------------------
            if (q.do_match) {
                const uint32_t last = cnt ? cnt - 1 : 0u;
                // guarded: lim can reach the sentinel value ~0 (narrow: only in the last tile; wide:
                // only if the tile's largest key is ~0 itself, else lim is clamped below it)
                const bool guarded = WIDE ? keyS[last] == ~0ull : tile == q.P - 1;
                // three items at a time, the loads of each search step issued together (the same loads
                // as one item after the other, but three dependency chains in flight per warp)
                constexpr int VX_EB = 3;
                static_assert(ITEMS % VX_EB == 0, "ITEMS must be a multiple of the phase-E batch");
#pragma unroll
                for (int g = 0; g < ITEMS; g += VX_EB) {
                    if (g * THREADS + wbase >= cnt) {   // warp-uniform: nothing of this batch is in range
#pragma unroll
                        for (int u = 0; u < VX_EB; u++) E[(g + u) * THREADS + tid] = 0u;
                        continue;
                    }
                    if (!guarded) {
                        uint64_t ki[VX_EB], lim[VX_EB], kn[VX_EB];
                        uint32_t pos[VX_EB];
#pragma unroll
                        for (int u = 0; u < VX_EB; u++) {
                            const uint32_t i = (g + u) * THREADS + tid;   // i + 7 < CAPA + 8: inside keyS
                            ki[u] = keyS[i];
                            kn[u] = keyS[i + 1];
                        }
#pragma unroll
                        for (int u = 0; u < VX_EB; u++) {
                            const uint32_t i = (g + u) * THREADS + tid;
                            const uint64_t kl = WIDE ? (ki[u] | q.lowmask) : ki[u];
                            uint64_t l = kl + Tm1;
                            if (WIDE && l < kl) l = ~0ull;
                            l = min(l, ki[u] | bmask);
                            if (WIDE) l = min(l, (uint64_t)(~0ull - 1ull));
                            lim[u] = l;
                            // the fast pass is valid iff the keys came out strictly increasing
                            if (!exact && i < cnt && kn[u] <= ki[u]) s_tie = 1u;
                            pos[u] = i;
                        }
                        // largest o in [0, 7] with key[i + o] <= lim (keys ascend; key[cnt] = ~0 > lim)
#pragma unroll
                        for (int u = 0; u < VX_EB; u++) kn[u] = keyS[pos[u] + 4];
#pragma unroll
                        for (int u = 0; u < VX_EB; u++) if (kn[u] <= lim[u]) pos[u] += 4;
#pragma unroll
                        for (int u = 0; u < VX_EB; u++) kn[u] = keyS[pos[u] + 2];
#pragma unroll
                        for (int u = 0; u < VX_EB; u++) if (kn[u] <= lim[u]) pos[u] += 2;
#pragma unroll
                        for (int u = 0; u < VX_EB; u++) kn[u] = keyS[pos[u] + 1];
#pragma unroll
                        for (int u = 0; u < VX_EB; u++) if (kn[u] <= lim[u]) pos[u] += 1;
#pragma unroll
                        for (int u = 0; u < VX_EB; u++) {
                            const uint32_t i = (g + u) * THREADS + tid;
                            uint32_t c = i < cnt ? pos[u] - i : 0u;
                            if (__any_sync(VX_FULL, c == 7u)) {
                                for (uint32_t j = i + 8;; j++) {
                                    const bool m = c >= 7u && j < cnt && keyS[min(j, last)] <= lim[u];
                                    c += m ? 1u : 0u;
                                    if (!__any_sync(VX_FULL, m)) break;
                                }
                            }
                            VX_CHECK(q.ctrl, i < (uint32_t)CAPA && (c == 0 || i + c < cnt));
                            E[i] = c;
                        }
                    } else {
#pragma unroll
                        for (int u = 0; u < VX_EB; u++) {
                            const uint32_t i = (g + u) * THREADS + tid;
                            const uint64_t ki = keyS[i];
                            const uint64_t kl = WIDE ? (ki | q.lowmask) : ki;
                            uint64_t lim = kl + Tm1;
                            if (lim < kl) lim = ~0ull;
                            lim = min(lim, ki | bmask);
                            uint32_t c = 0;
                            if (!exact && i < last && keyS[i + 1] <= ki) s_tie = 1u;
                            for (uint32_t j = i + 1;; j++) {
                                const bool m = i < cnt && j < cnt && keyS[min(j, last)] <= lim;
                                c += m ? 1u : 0u;
                                if (!__any_sync(VX_FULL, m)) break;
                            }
                            VX_CHECK(q.ctrl, i < (uint32_t)CAPA && (c == 0 || i + c < cnt));
                            E[i] = c;
                        }
                    }
                }
            }
            __syncthreads();
            if (!exact && s_tie) {                      // block-uniform: redo this tile exactly
                if (tid == 0) atomicAdd(&q.ctrl->retries, 1u);
                exact = 1u;
                continue;
            }
            break;
        }
        if (finished) break;

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

        if (q.do_match) {
            // ---- F. scan, publish the aggregate ---------------------------------------------------
            M = vx_block_exscan<THREADS, ITEMS>(E, s_warp);
            if (tid == 0) {
                E[CAPA] = M;
                if (tile) ((volatile unsigned long long *)q.status)[tile] = VX_ST_AGG | M;
            }
            __syncthreads();
        }
        // ---- G. sorted partition back in place; CSR offsets of Table 1 ---------------------------
#pragma unroll
        for (int it = 0; it < ITEMS; it++) {
            if (it * THREADS + wbase < cnt) {
                const uint32_t idx = it * THREADS + tid;
                if (idx < cnt) {
                    const uint64_t k = keyS[idx];
                    if constexpr (WIDE) {
                        const uint32_t b = nonS[idx];
                        reinterpret_cast<unsigned long long *>(src)[idx] = k;
                        src_b[idx] = (unsigned short)b;
                        // for the emit: nonce = (low pb key bits) << tile_log | the tile_log bits kept beside the key.
                        // pb <= 24, so only the LOW key word is needed and everything is 32-bit arithmetic
                        const uint32_t h = (uint32_t)k & (uint32_t)q.lowmask;
                        nonS[idx] = (h << q.nlo_bits) | b;
                        hiS[idx] = (uint8_t)(h >> (32u - q.nlo_bits));
                    } else {
                        src[idx] = make_uint4((uint32_t)k, (uint32_t)(k >> 32), nonS[idx], 0u);
                    }
                }
            }
        }
        const unsigned long long gb0 = (unsigned long long)tile << q.fb;
        const unsigned long long base1 = q.part_base[tile];
        for (uint32_t bl = tid; bl < nb_local; bl += THREADS) {
            const uint32_t s = bucket_start(bl), e = bucket_start(bl + 1);
            VX_CHECK(q.ctrl, s <= e && e <= cnt && gb0 + bl < q.NB && (!defer || bl < VX_DEFER_MAXB));
            cta_max_bucket = max(cta_max_bucket, e - s);
            q.t1_off[gb0 + bl] = base1 + s;
            if (defer) s_e2[bl] = E[s];
        }
        if (tile == q.P - 1 && tid == 0) q.t1_off[q.NB] = base1 + cnt;

        if (q.do_match) {
            if (defer) {
                pending = true;
                if (tid == 0) { s_p[0] = tile; s_p[1] = cnt; s_p[2] = M; }   // read behind the next tile's barriers
            } else {
                const unsigned long long base2 = lookback_emit(tile, cnt, M);
                for (uint32_t bl = tid; bl < nb_local; bl += THREADS)
                    q.t2_off[gb0 + bl] = base2 + E[bucket_start(bl)];
                if (tile == q.P - 1 && tid == 0) {
                    q.t2_off[q.NB] = base2 + M;
                    q.ctrl->t2_total = base2 + M;
                }
            }
        }
    }
    // largest bucket, one atomic per CTA
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) cta_max_bucket = max(cta_max_bucket, __shfl_xor_sync(VX_FULL, cta_max_bucket, d));
    if (lane == 0 && cta_max_bucket) atomicMax(&q.ctrl->max_bucket, cta_max_bucket);
}

// ------------------------------------------------------------------------------ warp-local variant
// vx_k_sort_match_wl: the same tile, the same phases A-C and the same arrays as vx_k_sort_match, but from the
// scatter on every WARP finishes its own share of the tile alone.  After phase C the records are grouped by bin
// and bins ascend with the hash, so warp w owns the bins [w * BPW, (w + 1) * BPW), BPW = bins / warps, i.e.
// the contiguous sorted positions [S, Send) = [bins[w * BPW], bins[(w + 1) * BPW]) -- a whole number of buckets
// when fb >= log2(warps), so no match crosses into another warp's range (matching is per bucket).
// The warp ranks its bins (D), counts its matches (E), scans them (F) and writes its records and bucket offsets
// back (G) behind __syncwarp only: the five CTA-wide barriers D|rewrite|E|F|F'|G of the classic kernel go, the
// warps of a CTA drift apart and fill each other's shared-memory latencies.  The tile total for the look-back
// is published by the last warp to finish its scan.  The Table-2 prefix E[] is relative to the warp's range;
// the warp's offset inside the tile is the sum of the totals of the warps before it, added in the emit (H),
// which the owning warp runs over its own range as well (deferred behind the next tile's phase A, as before).
// Applies to the narrow layout with matching on, log2(warps) <= fb <= 9 (K = 27 .. 32 at B = 24).  Same results
// bit for bit (tests/test_gpu_stage2_kernels.py runs every eligible geometry through both kernels).
// MEASURED AND NOT THE DEFAULT (DESIGN.md 6.2 "warp-local phases", profiles/r02_warp_local.md): K=31 33.9 ms
// against 30.0, K=32 71.2 against 64.7 -- 30 % more warp instructions (the bin-aligned runs of phase D, the
// dynamic loops) and the same share of barrier stalls, now all on the three barriers left (the warps' ranges
// differ by +-6 %, and the look-back wait grew).  Runs only with VX_OPT_STAGE2_KERNEL = 1.
template <int THREADS, int ITEMS, int BIN_BITS, int MINB>
__global__ void __launch_bounds__(THREADS, MINB)
vx_k_sort_match_wl(const __grid_constant__ VxS2Params q)
{
    constexpr uint32_t VX_NBINS = 1u << BIN_BITS;
    constexpr int CAPA = THREADS * ITEMS;
    constexpr int WARPS = THREADS / 32;
    constexpr uint32_t BPW = VX_NBINS / WARPS;          // bins per warp
    constexpr uint32_t VX_SCAN_L = 11;                  // positions per lane and round of the warp's scan (odd)
    extern __shared__ __align__(16) uint8_t vx_smem[];
    uint64_t *keyS = (uint64_t *)vx_smem;               // the layout of vx_k_sort_match
    uint32_t *nonS = (uint32_t *)(keyS + CAPA + 8);
    uint32_t *bins = nonS + CAPA;
    uint32_t *E = bins + VX_NBINS + 32;                 // match-count prefix, relative to the owning warp's range
    uint32_t *sub = E;                                  // phases C-D: ranking keys
    __shared__ uint32_t s_warp[32];
    __shared__ uint32_t s_tile, s_tie, s_cnt;
    __shared__ uint32_t s_done, s_M;                    // warps that have finished F; sum of their totals
    __shared__ uint32_t s_Mw[WARPS];                    // per-warp totals (read again by the deferred emit)
    __shared__ unsigned long long s_base2;
    constexpr uint32_t VX_DEFER_MAXB = 512;
    __shared__ uint32_t s_e2[VX_DEFER_MAXB];            // Table-2 prefix (warp-relative) at the first record of every bucket
    __shared__ uint32_t s_p[3];                         // tile, count, matches of the tile whose emit is pending

    const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
    const int sh = q.binshift - 32;
    const uint32_t submask = q.submask;
    const uint64_t Tm1 = q.Tm1;
    const uint64_t bmask = q.bmask;
    uint32_t cta_max_bucket = 0;
    const uint32_t nb_local = 1u << q.fb;
    const uint32_t nbw = nb_local / WARPS;              // buckets per warp (>= 1: checked at launch)
    const int bsh = BIN_BITS - (int)q.fb;               // first bin of local bucket bl = bl << bsh
    bool pending = false;
    uint32_t pS = 0, pEnd = 0;                          // the warp's range in the pending tile (warp-uniform)

    // ---- look-back for the Table-2 base, then H over the warp's own range
    auto lookback_emit = [&](uint32_t tile, uint32_t M) {
        if (tid < 32) {
            const unsigned long long b2 = vx_lookback(q.status, tile, M, lane);
            if (tid == 0) {
                s_base2 = b2;
                if (tile == q.tile_end - 1 && q.slice_end_out) *q.slice_end_out = b2 + M;
            }
        }
        __syncthreads();
        const unsigned long long base2 = s_base2;
        // totals of the warps before this one
        const uint32_t mw = lane < w ? s_Mw[lane] : 0u;
        const uint32_t Ow = __reduce_add_sync(VX_FULL, mw);
        if (base2 + M > q.t2_cap) {
            if (tid == 0) atomicOr(&q.ctrl->flags, VX_FLAG_T2_OVERFLOW);
        } else {
            const uint32_t Mw = s_Mw[w];
            uint2 *t2 = q.t2_rec + (base2 + Ow);
            for (uint32_t p0 = pS; p0 < pEnd; p0 += 32) {
                const uint32_t i = p0 + lane;
                uint32_t e0 = 0, c = 0;
                if (i < pEnd) {
                    e0 = E[i];
                    c = (i + 1 < pEnd ? E[i + 1] : Mw) - e0;
                    VX_CHECK(q.ctrl, e0 + c <= Mw && (c == 0 || i + c < pEnd) && base2 + Ow + e0 + c <= q.t2_cap);
                }
                const uint32_t cmax = __reduce_max_sync(VX_FULL, c);
                if (cmax) {
                    const uint32_t ni = nonS[min(i, (uint32_t)CAPA - 1u)];
                    const uint32_t *np = nonS + i + 1;
                    uint2 *dst = t2 + e0;
#pragma unroll
                    for (uint32_t t = 0; t < 4; t++)
                        if (t < c) dst[t] = make_uint2(ni, np[t]);
                    for (uint32_t t = 4; t < cmax; t++)
                        if (t < c) dst[t] = make_uint2(ni, np[t]);
                }
            }
        }
        const unsigned long long pg0 = (unsigned long long)tile << q.fb;
        for (uint32_t j = lane; j < nbw; j += 32) {
            const uint32_t bl = (uint32_t)w * nbw + j;
            q.t2_off[pg0 + bl] = base2 + Ow + s_e2[bl];
        }
        if (tile == q.P - 1 && tid == 0) {
            q.t2_off[q.NB] = base2 + M;
            q.ctrl->t2_total = base2 + M;
        }
    };

    for (;;) {
        // (no barrier here: a tile ends with one, and s_tile / s_cnt are read behind the next)
        if (tid == 0) {
            const uint32_t t = q.tile_begin + atomicAdd(&q.ctrl->ticket, 1u);
            s_tile = t;
            s_cnt = t < q.tile_end ? min(q.cursor[t], q.cap_check) : 0u;
            const uint32_t pf = t + gridDim.x;          // bulk L2 prefetch of a partition taken a round later
            if (pf < q.tile_end) {
                const uint32_t n = min(q.cursor[pf], q.cap_check);
                const char *p = reinterpret_cast<const char *>(q.part) + (size_t)pf * q.cap * 16;
                const uint32_t bytes = n * 16u;
                if (bytes) asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" :: "l"(p), "r"(bytes) : "memory");
            }
        }
        uint32_t exact = q.force_exact;
        uint32_t tile, cnt;
        uint32_t S = 0, Send = 0;
        bool finished = false;
        for (;;) {
            uint4 *src;
            uint64_t key[ITEMS];
            uint32_t non[ITEMS], sn[ITEMS];
            for (int i = tid; i < (int)(VX_NBINS + 32) / 4; i += THREADS)
                reinterpret_cast<uint4 *>(bins)[i] = make_uint4(0u, 0u, 0u, 0u);
            __syncthreads();
            if (tid == 0) { s_tie = 0u; s_done = 0u; s_M = 0u; }
            tile = s_tile;
            const bool valid = tile < q.tile_end;
            cnt = s_cnt;
            src = q.part + (size_t)tile * q.cap;
            // ---- A. load + bin count -----------------------------------------------------------
#pragma unroll
            for (int it = 0; it < ITEMS; it++) {
                const uint32_t idx = it * THREADS + tid;
                const uint4 r = idx < cnt ? __ldcs(src + idx) : make_uint4(0u, 0u, 0u, 0u);
                key[it] = ((uint64_t)r.y << 32) | r.x;
                non[it] = r.z;
            }
#pragma unroll
            for (int it = 0; it < ITEMS; it++) {
                const uint32_t idx = it * THREADS + tid;
                VX_CHECK(q.ctrl, cnt <= (uint32_t)CAPA && cnt <= q.cap && vx_bin<VX_NBINS>(key[it], sh) < VX_NBINS);
                if (idx < cnt) sn[it] = atomicAdd(&bins[vx_bin<VX_NBINS>(key[it], sh)], 1u);
            }
            if (pending) {                              // the previous tile of this CTA: look-back + H
                lookback_emit(s_p[0], s_p[2]);
                pending = false;
            }
            if (!valid) { finished = true; break; }
            __syncthreads();
            // ---- B. scan -------------------------------------------------------------------------
            {
                const uint32_t total = vx_block_exscan<THREADS, VX_NBINS / THREADS>(bins, s_warp);
                if (tid == 0) bins[VX_NBINS] = total;
            }
            __syncthreads();
            // ---- C. scatter to bin start + slot --------------------------------------------------
            {
                uint32_t pos[ITEMS];
#pragma unroll
                for (int it = 0; it < ITEMS; it++) {
                    const uint32_t idx = it * THREADS + tid;
                    pos[it] = idx < cnt ? bins[vx_bin<VX_NBINS>(key[it], sh)] + sn[it] : 0xffffffffu;
                }
#pragma unroll
                for (int it = 0; it < ITEMS; it++) {
                    if (pos[it] != 0xffffffffu) {
                        VX_CHECK(q.ctrl, pos[it] < cnt);
                        keyS[pos[it]] = key[it];
                        nonS[pos[it]] = non[it];
                        sub[pos[it]] = (vx_subkey(key[it], sh) & submask) | sn[it];
                        if (sn[it] > 15u) s_tie = 1u;   // a bin of more than 16 records: rank it exactly
                    }
                }
            }
            if (tid < 8) keyS[cnt + tid] = ~0ull;       // sentinels behind the last record
            __syncthreads();
            // a bin of more than 16 records: the slot no longer fits the ranking key's low bits, the fast ranks
            // could collide; nothing has been written yet -> the tile starts again with exact ranks
            if (!exact && s_tie) {
                if (tid == 0) atomicAdd(&q.ctrl->retries, 1u);
                exact = 1u;
                continue;
            }
            // ======== from here to the barrier at the end the warp works alone on [S, Send) ==========
            S = bins[(uint32_t)w * BPW];
            Send = bins[(uint32_t)w * BPW + BPW];
            VX_CHECK(q.ctrl, S <= Send && Send <= cnt);
            // ---- D. rank inside multi-record bins, a run of whole bins (<= 32 positions) at a time, in place
            {
                uint32_t b0 = (uint32_t)w * BPW, p0 = S;
                const uint32_t b_hi = b0 + BPW;
                while (b0 < b_hi) {                     // warp-uniform
                    // ends of the next 64 bins; the run takes those that end within 32 positions of p0
                    const uint32_t ia = b0 + 1 + lane, ib = ia + 32;
                    const uint32_t ea = ia <= b_hi ? bins[ia] : 0xffffffffu;
                    const uint32_t eb = ib <= b_hi ? bins[ib] : 0xffffffffu;
                    const uint32_t nb = __popc(__ballot_sync(VX_FULL, ea - p0 <= 32u)) +
                                        __popc(__ballot_sync(VX_FULL, eb - p0 <= 32u));
                    if (nb == 0) {
                        // a single bin of more than 32 records (never with real hashes): one lane sorts it by (H, n)
                        const uint32_t p1 = __shfl_sync(VX_FULL, ea, 0);
                        if (lane == 0) {
                            for (uint32_t a = p0 + 1; a < p1; a++) {
                                const uint64_t k = keyS[a];
                                const uint32_t nn = nonS[a];
                                uint32_t c = a;
                                while (c > p0 && (keyS[c - 1] > k || (keyS[c - 1] == k && nonS[c - 1] > nn))) {
                                    keyS[c] = keyS[c - 1]; nonS[c] = nonS[c - 1]; c--;
                                }
                                keyS[c] = k; nonS[c] = nn;
                            }
                        }
                        __syncwarp();
                        b0 += 1; p0 = p1;
                        continue;
                    }
                    const uint32_t p1 = nb <= 32u ? __shfl_sync(VX_FULL, ea, (nb - 1u) & 31u)
                                                  : __shfl_sync(VX_FULL, eb, (nb - 33u) & 31u);
                    const uint32_t i = p0 + lane;
                    const bool act = i < p1;
                    uint64_t k = 0ull;
                    uint32_t nn = 0u, s = 0u, n = 0u;
                    if (act) {
                        k = keyS[i];
                        nn = nonS[i];
                        const uint32_t b = vx_bin<VX_NBINS>(k, sh);
                        s = bins[b];
                        n = bins[b + 1] - s;
                        VX_CHECK(q.ctrl, b >= b0 && b < b0 + nb && s <= i && i < s + n && s + n <= p1);
                        if (n == 1u) n = 0u;            // alone in its bin: stays
                    }
                    const uint32_t nm = __reduce_max_sync(VX_FULL, n);
                    if (nm) {                           // warp-uniform: some bin of the run holds several records
                        uint32_t rank = 0;
                        if (!exact) {
                            const uint32_t *sp = sub + s;
                            const uint32_t ks = act ? sub[i] : 0u;
#pragma unroll
                            for (uint32_t j = 0; j < 4; j++) {
                                const uint32_t kj = j < n ? sp[j] : 0xffffffffu;
                                rank += kj < ks ? 1u : 0u;
                            }
                            if (nm > 4) {
#pragma unroll 1
                                for (uint32_t j = 4; j < nm; j++) {
                                    const uint32_t kj = j < n ? sp[j] : 0xffffffffu;
                                    rank += kj < ks ? 1u : 0u;
                                }
                            }
                        } else {                        // by (H, n), reading A10
                            const uint64_t *kp = keyS + s;
                            const uint32_t *np = nonS + s;
#pragma unroll 1
                            for (uint32_t j = 0; j < nm; j++)
                                if (j < n) rank += (kp[j] < k || (kp[j] == k && np[j] < nn)) ? 1u : 0u;
                        }
                        __syncwarp();                   // every lane has read its record and its bin
                        if (n) {
                            VX_CHECK(q.ctrl, s + rank < p1);
                            keyS[s + rank] = k;
                            nonS[s + rank] = nn;
                        }
                    }
                    b0 += nb; p0 = p1;
                }
            }
            __syncwarp();
            // ---- E. match count: lane i counts its successors within reach ------------------------
            {
                const uint32_t last = cnt ? cnt - 1 : 0u;
                const bool guarded = tile == q.P - 1;   // lim can reach the sentinel value ~0 only in the last tile
                constexpr int VX_EB = 3;
                for (uint32_t g0 = S; g0 < Send; g0 += 32u * VX_EB) {
                    if (!guarded) {
                        uint64_t ki[VX_EB], lim[VX_EB], kn[VX_EB];
                        uint32_t pos[VX_EB];
#pragma unroll
                        for (int u = 0; u < VX_EB; u++) {
                            // lanes behind the range read inside the arrays (results unused)
                            const uint32_t i = min(g0 + 32u * u + lane, (uint32_t)CAPA);
                            ki[u] = keyS[i];
                            kn[u] = keyS[i + 1];
                            pos[u] = i;
                        }
#pragma unroll
                        for (int u = 0; u < VX_EB; u++) {
                            lim[u] = min(ki[u] + Tm1, ki[u] | bmask);
                            // the fast pass is valid iff the keys came out strictly increasing (the first key of the
                            // next warp's range lies in a later bin: larger by construction)
                            if (!exact && pos[u] + 1 < Send && kn[u] <= ki[u]) s_tie = 1u;
                        }
#pragma unroll
                        for (int u = 0; u < VX_EB; u++) kn[u] = keyS[pos[u] + 4];
#pragma unroll
                        for (int u = 0; u < VX_EB; u++) if (kn[u] <= lim[u]) pos[u] += 4;
#pragma unroll
                        for (int u = 0; u < VX_EB; u++) kn[u] = keyS[pos[u] + 2];
#pragma unroll
                        for (int u = 0; u < VX_EB; u++) if (kn[u] <= lim[u]) pos[u] += 2;
#pragma unroll
                        for (int u = 0; u < VX_EB; u++) kn[u] = keyS[pos[u] + 1];
#pragma unroll
                        for (int u = 0; u < VX_EB; u++) if (kn[u] <= lim[u]) pos[u] += 1;
#pragma unroll
                        for (int u = 0; u < VX_EB; u++) {
                            const uint32_t i = g0 + 32u * u + lane;
                            uint32_t c = i < Send ? pos[u] - i : 0u;
                            if (__any_sync(VX_FULL, c == 7u)) {
                                for (uint32_t j = i + 8;; j++) {
                                    const bool m = c >= 7u && j < cnt && keyS[min(j, last)] <= lim[u];
                                    c += m ? 1u : 0u;
                                    if (!__any_sync(VX_FULL, m)) break;
                                }
                            }
                            VX_CHECK(q.ctrl, c == 0 || i + c < Send);
                            if (i < Send) E[i] = c;
                        }
                    } else {
#pragma unroll 1
                        for (int u = 0; u < VX_EB; u++) {
                            const uint32_t i = g0 + 32u * u + lane;
                            const bool in = i < Send;
                            const uint64_t ki = keyS[min(i, (uint32_t)CAPA)];
                            uint64_t lim = ki + Tm1;
                            if (lim < ki) lim = ~0ull;
                            lim = min(lim, ki | bmask);
                            uint32_t c = 0;
                            if (!exact && i + 1 < Send && keyS[i + 1] <= ki) s_tie = 1u;
                            for (uint32_t j = i + 1;; j++) {
                                const bool m = in && j < cnt && keyS[min(j, last)] <= lim;
                                c += m ? 1u : 0u;
                                if (!__any_sync(VX_FULL, m)) break;
                            }
                            VX_CHECK(q.ctrl, c == 0 || i + c < Send);
                            if (in) E[i] = c;
                        }
                    }
                }
            }
            __syncwarp();
            // ---- F. exclusive scan of the warp's counts, VX_SCAN_L consecutive positions per lane and round
            //         (an odd stride: conflict-free); the last warp to get here publishes the tile's total
            uint32_t Mw = 0;
            for (uint32_t base = S; base < Send; base += 32u * VX_SCAN_L) {
                const uint32_t n = min(Send - base, 32u * VX_SCAN_L);
                const uint32_t L = ((n + 31u) >> 5) | 1u;
                const uint32_t o = (uint32_t)lane * L;
                uint32_t v[VX_SCAN_L];
                uint32_t sum = 0;
#pragma unroll
                for (uint32_t kk = 0; kk < VX_SCAN_L; kk++) {
                    const uint32_t t = (kk < L && o + kk < n) ? E[base + o + kk] : 0u;
                    v[kk] = sum;
                    sum += t;
                }
                const uint32_t incl = vx_warp_incl_scan(sum, lane);
                const uint32_t off = Mw + incl - sum;
#pragma unroll
                for (uint32_t kk = 0; kk < VX_SCAN_L; kk++)
                    if (kk < L && o + kk < n) E[base + o + kk] = v[kk] + off;
                Mw += __shfl_sync(VX_FULL, incl, 31);
            }
            __syncwarp();
            if (lane == 0) {
                s_Mw[w] = Mw;
                atomicAdd(&s_M, Mw);
                __threadfence_block();
                if (atomicAdd(&s_done, 1u) == (uint32_t)WARPS - 1u) {
                    __threadfence_block();
                    const uint32_t M = *(volatile uint32_t *)&s_M;
                    // a tile that will be redone (its fast ranking met a tie) publishes nothing
                    if ((exact || *(volatile uint32_t *)&s_tie == 0u) && tile)
                        ((volatile unsigned long long *)q.status)[tile] = VX_ST_AGG | M;
                }
            }
            // ---- G. the warp's records back in place; CSR offsets of Table 1 for its buckets -----------
            for (uint32_t p = S + lane; p < Send; p += 32) {
                const uint64_t k = keyS[p];
                src[p] = make_uint4((uint32_t)k, (uint32_t)(k >> 32), nonS[p], 0u);
            }
            {
                const unsigned long long gb0 = (unsigned long long)tile << q.fb;
                const unsigned long long base1 = q.part_base[tile];
                for (uint32_t j = lane; j < nbw; j += 32) {
                    const uint32_t bl = (uint32_t)w * nbw + j;
                    const uint32_t s = bins[bl << bsh], e = bins[(bl + 1u) << bsh];
                    VX_CHECK(q.ctrl, S <= s && s <= e && e <= Send && gb0 + bl < q.NB && bl < VX_DEFER_MAXB);
                    cta_max_bucket = max(cta_max_bucket, e - s);
                    q.t1_off[gb0 + bl] = base1 + s;
                    s_e2[bl] = s < Send ? E[s] : Mw;
                }
                if (tile == q.P - 1 && tid == 0) q.t1_off[q.NB] = base1 + cnt;
            }
            __syncthreads();
            if (!exact && s_tie) {                      // block-uniform: redo this tile exactly
                if (tid == 0) atomicAdd(&q.ctrl->retries, 1u);
                exact = 1u;
                continue;
            }
            break;
        }
        if (finished) break;
        pending = true;
        pS = S; pEnd = Send;
        if (tid == 0) { s_p[0] = tile; s_p[1] = cnt; s_p[2] = s_M; }   // read behind the next tile's barriers
    }
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) cta_max_bucket = max(cta_max_bucket, __shfl_xor_sync(VX_FULL, cta_max_bucket, d));
    if (lane == 0 && cta_max_bucket) atomicMax(&q.ctrl->max_bucket, cta_max_bucket);
}

// ------------------------------------------------------------------------------ export
// Table-1 records [first, first + count) of the CSR numbering, gathered from the partition array
// into the external format nonce[NS] LE || hash[8] (digest bytes, = H big-endian) in `out`.
template <bool WIDE, int NS>
__global__ void __launch_bounds__(256)
vx_k_export_t1(const uint4 *__restrict__ part, const uint16_t *__restrict__ part_b,
               const unsigned long long *__restrict__ part_base, uint32_t P, uint32_t p_first, uint32_t cap,
               uint32_t pb, uint32_t nlo_bits,
               unsigned long long first, unsigned long long count, uint8_t *__restrict__ out)
{
    for (unsigned long long r = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; r < count;
         r += (unsigned long long)gridDim.x * blockDim.x) {
        const unsigned long long g = first + r;
        // partition holding CSR index g: the last p with part_base[p] <= g
        uint32_t lo = 0, hi = P;
        while (hi - lo > 1) {
            const uint32_t mid = (lo + hi) >> 1;
            if (part_base[mid] <= g) lo = mid; else hi = mid;
        }
        const size_t slot = (size_t)lo * cap + (g - part_base[lo]);
        unsigned long long H, n;
        if constexpr (WIDE) {
            const unsigned long long a = reinterpret_cast<const unsigned long long *>(part)[slot];
            H = pb ? ((unsigned long long)(lo + p_first) << (64 - pb)) | (a >> pb) : a;   // p_first: first partition of the pass
            n = ((a & ((1ull << pb) - 1ull)) << nlo_bits) | part_b[slot];
        } else {
            const uint4 rec = part[slot];
            H = ((unsigned long long)rec.y << 32) | rec.x;
            n = rec.z;
        }
        if constexpr (NS == 4) {
            uint32_t *o = reinterpret_cast<uint32_t *>(out) + 3 * r;
            o[0] = (uint32_t)n;
            o[1] = __byte_perm((uint32_t)(H >> 32), 0, 0x0123);
            o[2] = __byte_perm((uint32_t)H, 0, 0x0123);
        } else {
            uint8_t *o = out + (size_t)(NS + 8) * r;
#pragma unroll
            for (int j = 0; j < NS; j++) o[j] = (uint8_t)(n >> (8 * j));
#pragma unroll
            for (int j = 0; j < 8; j++) o[NS + j] = (uint8_t)(H >> (8 * (7 - j)));
        }
    }
}

// wide Table-2 records [first, first + count) -> external nonce1[5] || nonce2[5], little-endian
__global__ void __launch_bounds__(256)
vx_k_export_t2(const uint2 *__restrict__ rec, const uint8_t *__restrict__ hi, unsigned long long first,
               unsigned long long count, uint8_t *__restrict__ out)
{
    for (unsigned long long r = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; r < count;
         r += (unsigned long long)gridDim.x * blockDim.x) {
        const uint2 v = rec[first + r];
        const uint8_t h = hi[first + r];
        uint8_t *o = out + 10 * r;
#pragma unroll
        for (int j = 0; j < 4; j++) { o[j] = (uint8_t)(v.x >> (8 * j)); o[5 + j] = (uint8_t)(v.y >> (8 * j)); }
        o[4] = h & 15u;
        o[9] = h >> 4;
    }
}

// re-keyed Table 2 (8(f2)): the partition array holds {H2, pair index} sorted by H2; records
// [first, first + count) of its CSR numbering are the pairs t2_rec[index], gathered here.
__global__ void __launch_bounds__(256)
vx_k_export_rekey(const uint4 *__restrict__ part, const unsigned long long *__restrict__ part_base, uint32_t P,
                  uint32_t cap, const uint2 *__restrict__ t2_rec, unsigned long long first,
                  unsigned long long count, uint2 *__restrict__ out)
{
    for (unsigned long long r = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; r < count;
         r += (unsigned long long)gridDim.x * blockDim.x) {
        const unsigned long long g = first + r;
        uint32_t lo = 0, hi = P;
        while (hi - lo > 1) {
            const uint32_t mid = (lo + hi) >> 1;
            if (part_base[mid] <= g) lo = mid; else hi = mid;
        }
        const uint4 rec = part[(size_t)lo * cap + (g - part_base[lo])];
        out[r] = t2_rec[rec.z];
    }
}

// the same in the wide layout: pair index = (low pb bits of a) << 16 | b; the pair comes from the packed
// Table 2 and leaves in the external format, nonce1[NS] || nonce2[NS]
template <int NS>
__global__ void __launch_bounds__(256)
vx_k_export_rekey_wide(const unsigned long long *__restrict__ part_a, const uint16_t *__restrict__ part_b,
                       const unsigned long long *__restrict__ part_base, uint32_t P, uint32_t cap, uint32_t pb,
                       const uint2 *__restrict__ t2_rec, const uint8_t *__restrict__ t2_hi,
                       unsigned long long first, unsigned long long count, uint8_t *__restrict__ out)
{
    for (unsigned long long r = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; r < count;
         r += (unsigned long long)gridDim.x * blockDim.x) {
        const unsigned long long g = first + r;
        uint32_t lo = 0, hi = P;
        while (hi - lo > 1) {
            const uint32_t mid = (lo + hi) >> 1;
            if (part_base[mid] <= g) lo = mid; else hi = mid;
        }
        const size_t slot = (size_t)lo * cap + (g - part_base[lo]);
        const unsigned long long idx = ((part_a[slot] & ((1ull << pb) - 1ull)) << 16) | part_b[slot];
        const uint2 v = t2_rec[idx];
        if constexpr (NS == 4) {
            reinterpret_cast<uint2 *>(out)[r] = v;
        } else {
            const uint8_t h = t2_hi[idx];
            uint8_t *o = out + 10 * r;
#pragma unroll
            for (int j = 0; j < 4; j++) { o[j] = (uint8_t)(v.x >> (8 * j)); o[5 + j] = (uint8_t)(v.y >> (8 * j)); }
            o[4] = h & 15u;
            o[9] = h >> 4;
        }
    }
}

cudaError_t vx_launch_export_rekey(const VxGeom &g, uint8_t *ws, uint64_t first, uint64_t count, cudaStream_t st)
{
    if (count == 0) return cudaSuccess;
    uint64_t grid = (count + 255) / 256;
    if (grid > (uint64_t)vx_sm_count() * 16) grid = (uint64_t)vx_sm_count() * 16;
    const unsigned long long *pbase = (const unsigned long long *)(ws + g.off_part_base);
    if (g.wide) {
        const unsigned long long *pa = (const unsigned long long *)(ws + g.off_part);
        const uint16_t *pbb = (const uint16_t *)(ws + g.off_part_b);
        if (g.nonce_size == 5)
            vx_k_export_rekey_wide<5><<<(unsigned)grid, 256, 0, st>>>(pa, pbb, pbase, (uint32_t)g.P, g.cap, g.pb,
                (const uint2 *)(ws + g.off_t2_rec), ws + g.off_t2_hi, first, count, ws + g.off_stage);
        else
            vx_k_export_rekey_wide<4><<<(unsigned)grid, 256, 0, st>>>(pa, pbb, pbase, (uint32_t)g.P, g.cap, g.pb,
                (const uint2 *)(ws + g.off_t2_rec), ws + g.off_t2_hi, first, count, ws + g.off_stage);
        return cudaGetLastError();
    }
    vx_k_export_rekey<<<(unsigned)grid, 256, 0, st>>>((const uint4 *)(ws + g.off_part), pbase, (uint32_t)g.P,
                                                      g.cap, (const uint2 *)(ws + g.off_t2_rec), first, count,
                                                      (uint2 *)(ws + g.off_stage));
    return cudaGetLastError();
}

cudaError_t vx_launch_export_t1(const VxGeom &g, uint8_t *ws, uint64_t first, uint64_t count,
                                cudaStream_t st)
{
    if (count == 0) return cudaSuccess;
    uint64_t grid = (count + 255) / 256;
    if (grid > (uint64_t)vx_sm_count() * 16) grid = (uint64_t)vx_sm_count() * 16;
    const uint4 *part = (const uint4 *)(ws + g.off_part);
    const uint16_t *part_b = (const uint16_t *)(ws + g.off_part_b);
    const unsigned long long *pbase = (const unsigned long long *)(ws + g.off_part_base);
    uint8_t *out = ws + g.off_stage;
    if (g.nonce_size == 5)
        vx_k_export_t1<true, 5><<<(unsigned)grid, 256, 0, st>>>(part, part_b, pbase, (uint32_t)g.P, (uint32_t)g.p_first, g.cap, g.pb, g.tile_log, first, count, out);
    else if (g.wide)
        vx_k_export_t1<true, 4><<<(unsigned)grid, 256, 0, st>>>(part, part_b, pbase, (uint32_t)g.P, (uint32_t)g.p_first, g.cap, g.pb, g.tile_log, first, count, out);
    else
        vx_k_export_t1<false, 4><<<(unsigned)grid, 256, 0, st>>>(part, part_b, pbase, (uint32_t)g.P, (uint32_t)g.p_first, g.cap, g.pb, g.tile_log, first, count, out);
    return cudaGetLastError();
}

cudaError_t vx_launch_export_t2(const VxGeom &g, uint8_t *ws, uint64_t first, uint64_t count,
                                cudaStream_t st, size_t stage_offset)
{
    if (count == 0) return cudaSuccess;
    uint64_t grid = (count + 255) / 256;
    if (grid > (uint64_t)vx_sm_count() * 16) grid = (uint64_t)vx_sm_count() * 16;
    vx_k_export_t2<<<(unsigned)grid, 256, 0, st>>>((const uint2 *)(ws + g.off_t2_rec), ws + g.off_t2_hi,
                                                   first, count, ws + g.off_stage + stage_offset);
    return cudaGetLastError();
}

size_t vx_stage2_smem_bytes(const VxGeom &g)
{
    const size_t CAPA = g.tile_log == VX_TILE_LOG_BIG ? (size_t)VX_S2B_THREADS * VX_S2B_ITEMS
                                                      : (size_t)VX_S2_THREADS * VX_S2_ITEMS;
    const size_t nbins = (size_t)1 << g.tile_log;
    return (CAPA + 8) * 8 + CAPA * 4 + (nbins + 32) * 4 + (CAPA + 32) * 4 + (g.wide ? CAPA + 16 : 0);
}

#define VX_S2_KERNEL(WIDE) vx_k_sort_match<VX_S2_THREADS, VX_S2_ITEMS, VX_TILE_LOG, VX_S2_MINB, WIDE>
#define VX_S2B_KERNEL(WIDE) vx_k_sort_match<VX_S2B_THREADS, VX_S2B_ITEMS, VX_TILE_LOG_BIG, 1, WIDE>
#define VX_S2_KERNEL_WL vx_k_sort_match_wl<VX_S2_THREADS, VX_S2_ITEMS, VX_TILE_LOG, VX_S2_MINB>
#define VX_S2B_KERNEL_WL vx_k_sort_match_wl<VX_S2B_THREADS, VX_S2B_ITEMS, VX_TILE_LOG_BIG, 1>

// the warp-local kernel applies when every warp's share of the bins is a whole number of buckets (no match
// crosses a warp's range), the bucket starts are bin starts and the deferred emit's bucket table fits
bool vx_stage2_warp_local(const VxGeom &g, bool do_match)
{
    const uint32_t warps_log = g.tile_log == VX_TILE_LOG_BIG ? 5u : 4u;   // 1024 / 512 threads
    return do_match && !g.wide && g.s2_kernel == 1u && g.fb >= warps_log && g.fb <= 9u;
}

cudaError_t vx_stage2_configure(void)
{
    VxGeom g{};
    g.tile_log = VX_TILE_LOG;
    const int small = (int)vx_stage2_smem_bytes(g);
    g.tile_log = VX_TILE_LOG_BIG;
    const int big = (int)vx_stage2_smem_bytes(g);
    g.wide = 1;                                         // + the emit's byte of high nonce bits per record
    const int big_wide = (int)vx_stage2_smem_bytes(g);
    g.tile_log = VX_TILE_LOG;
    const int small_wide = (int)vx_stage2_smem_bytes(g);
    cudaError_t e = cudaFuncSetAttribute(VX_S2_KERNEL(false), cudaFuncAttributeMaxDynamicSharedMemorySize, small);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(VX_S2_KERNEL(true), cudaFuncAttributeMaxDynamicSharedMemorySize, small_wide);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(VX_S2B_KERNEL(false), cudaFuncAttributeMaxDynamicSharedMemorySize, big);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(VX_S2B_KERNEL(true), cudaFuncAttributeMaxDynamicSharedMemorySize, big_wide);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(VX_S2_KERNEL_WL, cudaFuncAttributeMaxDynamicSharedMemorySize, small);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(VX_S2B_KERNEL_WL, cudaFuncAttributeMaxDynamicSharedMemorySize, big);
    return e;
}

cudaError_t vx_launch_stage2(const VxGeom &g, uint8_t *ws, bool do_match, bool force_exact, int num_sms,
                             cudaStream_t st, uint32_t tile_begin, uint32_t tile_end,
                             unsigned long long *slice_end_out)
{
    VxCtrl *ctrl = (VxCtrl *)(ws + g.off_ctrl);
    if (tile_end > g.P) tile_end = (uint32_t)g.P;
    if (tile_begin >= tile_end) return cudaErrorInvalidValue;
    // ticket; for the first (or only) slice of the plot also the largest-bucket word and the look-back state
    const bool first = tile_begin == 0;
    cudaError_t e = vx_launch_clear(st, first ? ws + g.off_status : nullptr, first ? g.P * sizeof(unsigned long long) : 0,
                                    nullptr, 0, &ctrl->ticket, first ? &ctrl->max_bucket : nullptr);
    if (e != cudaSuccess) return e;
    VxS2Params q;
    q.part = (uint4 *)(ws + g.off_part);
    q.cursor = (const uint32_t *)(ws + g.off_cursor);
    q.part_base = (const unsigned long long *)(ws + g.off_part_base);
    q.status = (unsigned long long *)(ws + g.off_status);
    q.ctrl = ctrl;
    q.t1_off = (unsigned long long *)(ws + g.off_t1_off);
    q.t2_rec = (uint2 *)(ws + g.off_t2_rec);
    q.t2_off = (unsigned long long *)(ws + g.off_t2_off);
    q.N = g.N; q.NB = g.NBp; q.t2_cap = g.t2_check;      // bucket indices in the kernel are relative to the pass
    q.P = (uint32_t)g.P; q.cap = g.cap; q.cap_check = g.cap_check; q.pb = g.pb; q.fb = g.fb; q.K = g.K; q.B = g.B;
    q.do_match = do_match ? 1u : 0u;
    q.force_exact = force_exact ? 1u : 0u;
    // 28 hash bits at most: the low 4 bits of the ranking key hold the record's slot in its bin
    q.submask = g.subkey_bits >= 28 ? 0xfffffff0u : g.subkey_bits == 0 ? 0u : ~0u << (32 - g.subkey_bits);
    q.tile_begin = tile_begin; q.tile_end = tile_end; q.slice_end_out = slice_end_out;
    if (g.pb + g.tile_log > 32 && !g.wide) return cudaErrorInvalidValue;   // bin and sub-key sit in the high word
    q.part_b = (uint16_t *)(ws + g.off_part_b);
    q.t2_hi = ws + g.off_t2_hi;
    // sort-key geometry.  narrow: key = H.  wide: key = a = (H << pb) | (n >> 12)
    const unsigned long long T = 1ull << (64 - g.K);
    if (g.wide) {
        q.binshift = 64 - (int)g.tile_log;
        q.bshift = 64 - (int)g.fb;                      // only used when fb > VX_BIN_BITS (then < 64)
        q.lowmask = (1ull << g.pb) - 1ull;
        q.Tm1 = (T - 1ull) << g.pb;
        q.bmask = g.fb ? (1ull << (64 - g.fb)) - 1ull : ~0ull;
    } else {
        q.binshift = 64 - (int)g.pb - (int)g.tile_log;
        q.bshift = 64 - (int)g.B;
        q.lowmask = 0ull;
        q.Tm1 = T - 1ull;
        q.bmask = (1ull << q.bshift) - 1ull;
    }
    const size_t smem = vx_stage2_smem_bytes(g);
    q.nlo_bits = g.tile_log;
    const bool big = g.tile_log == VX_TILE_LOG_BIG;
    uint64_t grid = (uint64_t)num_sms * (big ? 1 : VX_S2_MINB);
#ifdef VX_EXP_GRID_PER_SM
    // measurement only (DESIGN.md 6.2 "what bounds it"): VX_NVCC_EXTRA=-DVX_EXP_GRID_PER_SM=1 runs the fused
    // kernel with one resident tile per SM; never defined in the product build
    grid = (uint64_t)num_sms * VX_EXP_GRID_PER_SM;
#endif
    if (grid > tile_end - tile_begin) grid = tile_end - tile_begin;
    if (vx_stage2_warp_local(g, do_match)) {
        if (big) VX_S2B_KERNEL_WL<<<(unsigned)grid, VX_S2B_THREADS, smem, st>>>(q);
        else VX_S2_KERNEL_WL<<<(unsigned)grid, VX_S2_THREADS, smem, st>>>(q);
    }
    else if (big && g.wide) VX_S2B_KERNEL(true)<<<(unsigned)grid, VX_S2B_THREADS, smem, st>>>(q);
    else if (big) VX_S2B_KERNEL(false)<<<(unsigned)grid, VX_S2B_THREADS, smem, st>>>(q);
    else if (g.wide) VX_S2_KERNEL(true)<<<(unsigned)grid, VX_S2_THREADS, smem, st>>>(q);
    else VX_S2_KERNEL(false)<<<(unsigned)grid, VX_S2_THREADS, smem, st>>>(q);
    return cudaGetLastError();
}
