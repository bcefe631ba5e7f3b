// vx_stage1.cu -- stage 1 of the plot: BLAKE3 keyed hash of every nonce + scatter of the
// (nonce, H) record into its hash-prefix partition in HBM.
//
// PAPER.md L81 (III-A): "a custom Blake3 CUDA kernel launches one thread per nonce across the full
// 2^k nonce space, hashing each nonce independently and inserting the resulting nonce-hash pair
// into its corresponding bucket in GPU VRAM using atomic operations"; L91 (III-B): "atomically
// claims a slot in the corresponding bucket using atomicAdd".  SURVEY.md 8(a) rows a1-a5.
//
// What differs from the paper's kernel: the atomic append targets 2^pb
// coarse partitions (pb = K - 12), not 2^24 buckets, so the set of partially written 32-byte
// sectors (one per partition) stays far below the 126 MB L2 and is merged there; a record is ONE
// aligned 16-byte store {H, nonce} because scattered stores on B200 are bound by request count
// (~50 G/s once the write frontier spans more pages than the TLB reaches), not by bytes;
// several nonces per thread keep the atomics' latency off the ALU pipe.
#include "vx_internal.h"

#define VX_S1_THREADS 256
#define VX_S1_NPT 4

// The record is one aligned 16-byte store {H lo, H hi, nonce lo, nonce hi}.  The wide layout
// (K >= 33) runs this same kernel per round into its scratch partitions (vx_k_compact below).
template <bool NONCE5>
__global__ void __launch_bounds__(VX_S1_THREADS)
vx_k_hash_scatter(const __grid_constant__ VxHashConst hc, uint64_t n_begin, uint64_t N, uint32_t pb, uint32_t cap,
                  uint32_t cap_check, uint32_t p_first, uint32_t p_count, uint4 *__restrict__ part,
                  uint32_t *__restrict__ cursor, VxCtrl *__restrict__ ctrl)
{
    // p_first, p_count: the partitions this pass keeps (all 2^pb of them unless the plot is made in
    // bucket-range passes); a record of any other partition is hashed and dropped
    // nonces [n_begin, N): the whole plot, or one round of it (wide layout, vx_launch_stage1)
    const uint64_t base = n_begin + (uint64_t)blockIdx.x * (VX_S1_THREADS * VX_S1_NPT) + threadIdx.x;
    uint64_t H[VX_S1_NPT];
#pragma unroll
    for (int k = 0; k < VX_S1_NPT; k++) {
        const uint64_t n = base + (uint64_t)k * VX_S1_THREADS;
        H[k] = vx_blake3_h<NONCE5>(hc, (uint32_t)n, (uint32_t)(n >> 32));
    }
#pragma unroll
    for (int k = 0; k < VX_S1_NPT; k++) {
        const uint64_t n = base + (uint64_t)k * VX_S1_THREADS;
        if (n < N) {
            const uint32_t p = (pb ? (uint32_t)(H[k] >> (64 - pb)) : 0u) - p_first;
            if (p >= p_count) continue;
            VX_CHECK(ctrl, pb == 0 || p + p_first < (1u << pb));
            const uint32_t slot = atomicAdd(&cursor[p], 1u);
            if (slot < cap_check) {                     // = cap, unless a test lowered it
                VX_CHECK(ctrl, slot < cap);
                // one 16-byte store per record: scattered stores are bound by requests, not bytes
                part[(uint64_t)p * cap + slot] =
                    make_uint4((uint32_t)H[k], (uint32_t)(H[k] >> 32), (uint32_t)n, (uint32_t)(n >> 32));
            } else {
                atomicOr(&ctrl->flags, VX_FLAG_PART_OVERFLOW);
            }
        }
    }
}

// ----------------------------------------------------------------------------- one plot over G GPUs
// SURVEY.md 8(e) / 8(f4) (the paper's boxes hold 8 GPUs, it uses one): rank r hashes
// the nonces [r 2^K / G, (r + 1) 2^K / G); buckets are owned by hash range -- rank g owns the
// partitions (and buckets) whose top log2 G hash bits are g -- and the record goes straight from the
// hashing thread to its owner: the slot is claimed with an atomic on the OWNER's cursor and the
// 16-byte record stored into the OWNER's partition array, both through peer pointers (NVLink 5 /
// NVSwitch peer stores: the all-to-all is fused with the first partition pass, nothing is staged
// or sent twice).  Every rank's workspace has the same carve-up (one "pass" of a plot created with
// VX_CREATE_PASSES_LOG(log2 G)), so a peer is addressed by its workspace base alone.
struct VxPeers { uint8_t *ws[VX_MAX_SHARD_WORLD]; };

__global__ void __launch_bounds__(VX_S1_THREADS)
vx_k_hash_scatter_sharded(const __grid_constant__ VxHashConst hc, const __grid_constant__ VxPeers peers,
                          uint64_t n_begin, uint64_t n_end, uint32_t pb, uint32_t own_shift, uint32_t cap,
                          uint32_t cap_check, size_t off_part, size_t off_cursor, size_t off_ctrl)
{
    const uint64_t base = n_begin + (uint64_t)blockIdx.x * (VX_S1_THREADS * VX_S1_NPT) + threadIdx.x;
    uint64_t H[VX_S1_NPT];
#pragma unroll
    for (int k = 0; k < VX_S1_NPT; k++) {
        const uint64_t n = base + (uint64_t)k * VX_S1_THREADS;
        H[k] = vx_blake3_h<false>(hc, (uint32_t)n, (uint32_t)(n >> 32));
    }
#pragma unroll
    for (int k = 0; k < VX_S1_NPT; k++) {
        const uint64_t n = base + (uint64_t)k * VX_S1_THREADS;
        if (n < n_end) {
            const uint32_t p = (uint32_t)(H[k] >> (64 - pb));          // global partition (pb >= log2 G >= 1)
            const uint32_t owner = p >> own_shift;                     // its top log2 G bits
            const uint32_t pl = p & ((1u << own_shift) - 1u);          // partition index at the owner
            uint8_t *ws = peers.ws[owner];
            const uint32_t slot = atomicAdd(reinterpret_cast<uint32_t *>(ws + off_cursor) + pl, 1u);
            if (slot < cap_check)
                reinterpret_cast<uint4 *>(ws + off_part)[(uint64_t)pl * cap + slot] =
                    make_uint4((uint32_t)H[k], (uint32_t)(H[k] >> 32), (uint32_t)n, (uint32_t)(n >> 32));
            else
                atomicOr(&reinterpret_cast<VxCtrl *>(ws + off_ctrl)->flags, VX_FLAG_PART_OVERFLOW);
        }
    }
}

// ----------------------------------------------------------------------------- wide: compaction
// Stage 1 in rounds (wide layout, K >= 33).  A 10-byte record written
// straight from the hash kernel costs two scattered store requests plus the atomic, and scattered
// stores are bound by requests: K=33 stage 1 ran 2.6x over its ALU bound that way.  Instead each
// round scatters its slice as 16-byte records (ONE request each, the narrow kernel above) into
// 2^pb_tmp scratch partitions, and this kernel moves every scratch partition into the 2^d final
// partitions it covers (d = pb - pb_tmp) in the compact layout a = (H << pb) | (n >> nlo_bits),
// b = n & (2^nlo_bits - 1): contiguous 16-byte loads, and stores that are contiguous per final
// partition, so this pass runs at HBM speed (26 bytes per record).
// One CTA per scratch partition; it is the only writer of its final partitions' cursors in this
// round (rounds are serialised on the stream), so those are plain loads and stores.
#define VX_CP_THREADS 256
#define VX_CP_MAXSUB 4
__global__ void __launch_bounds__(VX_CP_THREADS)
vx_k_compact(const uint4 *__restrict__ tmp, uint32_t *__restrict__ cursor_tmp, uint32_t cap_tmp,
             uint32_t pb, uint32_t d, uint32_t nlo_bits, uint32_t cap, uint32_t cap_check,
             unsigned long long *__restrict__ part_a, uint16_t *__restrict__ part_b,
             uint32_t *__restrict__ cursor, VxCtrl *__restrict__ ctrl)
{
    __shared__ uint32_t s_base[VX_CP_MAXSUB], s_cnt[VX_CP_MAXSUB];
    const uint32_t p = blockIdx.x, tid = threadIdx.x, lane = tid & 31;
    const uint32_t nsub = 1u << d;
    const uint32_t cnt_raw = cursor_tmp[p];
    const uint32_t cnt = min(cnt_raw, cap_tmp);
    // (p and the final partitions (p << d) + s are indices within the pass; the low d bits of the
    // global partition index H >> (64 - pb) are those of the local one: a pass starts on a multiple of 2^d)
    if (tid < nsub) { s_base[tid] = cursor[(p << d) + tid]; s_cnt[tid] = 0u; }
    if (tid == 0 && cnt_raw > cap_tmp) atomicOr(&ctrl->flags, VX_FLAG_PART_OVERFLOW);
    __syncthreads();
    const uint4 *src = tmp + (size_t)p * cap_tmp;
    bool over = false;
    for (uint32_t i0 = 0; i0 < cnt; i0 += VX_CP_THREADS) {
        const uint32_t i = i0 + tid;
        const bool valid = i < cnt;
        const uint4 r = valid ? __ldcs(src + i) : make_uint4(0u, 0u, 0u, 0u);
        const unsigned long long H = ((unsigned long long)r.y << 32) | r.x;
        const unsigned long long n = ((unsigned long long)r.w << 32) | r.z;
        const uint32_t s = d ? (uint32_t)(H >> (64 - pb)) & (nsub - 1u) : 0u;
        // warp-aggregated slot claim, one shared atomic per (warp, final partition)
        const unsigned peers = __match_any_sync(0xffffffffu, valid ? s : 0xffffffffu);
        const int leader = __ffs(peers) - 1;
        uint32_t off = 0;
        if (valid && (int)lane == leader) off = atomicAdd(&s_cnt[s], (uint32_t)__popc(peers));
        off = __shfl_sync(0xffffffffu, off, leader);
        if (valid) {
            const uint32_t slot = s_base[s] + off + __popc(peers & ((1u << lane) - 1u));
            VX_CHECK(ctrl, s < nsub && nsub <= VX_CP_MAXSUB);
            if (slot < cap_check) {
                const size_t at = (size_t)((p << d) + s) * cap + slot;
                VX_CHECK(ctrl, slot < cap && ((p << d) + s) < gridDim.x << d);
                part_a[at] = (H << pb) | (n >> nlo_bits);
                part_b[at] = (uint16_t)(n & ((1u << nlo_bits) - 1u));
            } else {
                over = true;
            }
        }
    }
    if (over) atomicOr(&ctrl->flags, VX_FLAG_PART_OVERFLOW);
    __syncthreads();
    if (tid < nsub) cursor[(p << d) + tid] = s_base[tid] + s_cnt[tid];   // counts every claim, like stage 1's atomics
    if (tid == 0) cursor_tmp[p] = 0u;                   // ready for the next round (read above, before the first barrier)
}

// Zeroes up to two regions (16-byte granules; every workspace region is 256-byte aligned and padded)
// and up to two single words.  A kernel rather than cudaMemsetAsync: a memset may be handed to a copy
// engine, where it queues behind another plot's gigabyte-sized Table-2 copies (vx_egress.cu) and
// holds this plot's kernels back until they drain.
__global__ void __launch_bounds__(256)
vx_k_clear(uint4 *__restrict__ a, size_t na, uint4 *__restrict__ b, size_t nb, uint32_t *w0, uint32_t *w1)
{
    const size_t i0 = (size_t)blockIdx.x * blockDim.x + threadIdx.x, step = (size_t)gridDim.x * blockDim.x;
    for (size_t i = i0; i < na; i += step) a[i] = make_uint4(0u, 0u, 0u, 0u);
    for (size_t i = i0; i < nb; i += step) b[i] = make_uint4(0u, 0u, 0u, 0u);
    if (i0 == 0) { if (w0) *w0 = 0u; if (w1) *w1 = 0u; }
}

cudaError_t vx_launch_clear(cudaStream_t st, void *a, size_t bytes_a, void *b, size_t bytes_b, uint32_t *w0, uint32_t *w1)
{
    const size_t na = (bytes_a + 15) / 16, nb = (bytes_b + 15) / 16;
    size_t grid = ((na > nb ? na : nb) + 255) / 256;
    if (grid < 1) grid = 1;
    const size_t gmax = (size_t)vx_sm_count() * 8;
    if (grid > gmax) grid = gmax;
    vx_k_clear<<<(unsigned)grid, 256, 0, st>>>((uint4 *)a, na, (uint4 *)b, nb, w0, w1);
    return cudaGetLastError();
}

// Exclusive prefix sum of the clamped partition counts: part_base[p] = number of records in
// partitions < p, part_base[P] = total.  One CTA; P <= 2^20 so this is a few tens of microseconds.
#define VX_SCAN_THREADS 1024
#define VX_SCAN_ITEMS 16
__global__ void __launch_bounds__(VX_SCAN_THREADS)
vx_k_partition_scan(const uint32_t *__restrict__ cursor, uint32_t cap, uint64_t P,
                    unsigned long long *__restrict__ part_base)
{
    __shared__ unsigned long long s_warp[32];
    __shared__ unsigned long long s_carry;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid == 0) s_carry = 0;
    __syncthreads();
    for (uint64_t chunk = 0; chunk < P; chunk += (uint64_t)VX_SCAN_THREADS * VX_SCAN_ITEMS) {
        const uint64_t i0 = chunk + (uint64_t)tid * VX_SCAN_ITEMS;
        uint32_t c[VX_SCAN_ITEMS];
        unsigned long long sum = 0;
#pragma unroll
        for (int k = 0; k < VX_SCAN_ITEMS; k++) {
            c[k] = (i0 + k < P) ? min(cursor[i0 + k], cap) : 0u;
            sum += c[k];
        }
        unsigned long long incl = sum;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const unsigned long long o = __shfl_up_sync(0xffffffffu, incl, d);
            if (lane >= d) incl += o;
        }
        if (lane == 31) s_warp[warp] = incl;
        __syncthreads();
        unsigned long long wbase = 0, total = 0;
        {
            unsigned long long w = s_warp[lane];   // 32 warps exactly
            unsigned long long wi = w;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                const unsigned long long o = __shfl_up_sync(0xffffffffu, wi, d);
                if (lane >= d) wi += o;
            }
            wbase = __shfl_sync(0xffffffffu, wi - w, warp);
            total = __shfl_sync(0xffffffffu, wi, 31);
        }
        unsigned long long run = s_carry + wbase + (incl - sum);
#pragma unroll
        for (int k = 0; k < VX_SCAN_ITEMS; k++) {
            if (i0 + k < P) part_base[i0 + k] = run;
            run += c[k];
        }
        __syncthreads();
        if (tid == 0) s_carry += total;
        __syncthreads();
    }
    if (tid == 0) part_base[P] = s_carry;
}

// ----------------------------------------------------------------------------- hash alone
template <bool NONCE5>
__global__ void __launch_bounds__(VX_S1_THREADS)
vx_k_hash_range(const __grid_constant__ VxHashConst hc, uint64_t nonce_begin, uint64_t count,
                uint64_t *__restrict__ out)
{
    const uint64_t i = (uint64_t)blockIdx.x * VX_S1_THREADS + threadIdx.x;
    if (i < count) {
        const uint64_t n = nonce_begin + i;
        out[i] = vx_blake3_h<NONCE5>(hc, (uint32_t)n, (uint32_t)(n >> 32));
    }
}

// the BLAKE3 stage with no table traffic: xor-fold of every hash into one word per CTA
template <bool NONCE5>
__global__ void __launch_bounds__(VX_S1_THREADS)
vx_k_hash_sink(const __grid_constant__ VxHashConst hc, uint64_t count, uint64_t *__restrict__ sink)
{
    const uint64_t base = (uint64_t)blockIdx.x * (VX_S1_THREADS * VX_S1_NPT) + threadIdx.x;
    uint64_t x = 0;
#pragma unroll
    for (int k = 0; k < VX_S1_NPT; k++) {
        const uint64_t n = base + (uint64_t)k * VX_S1_THREADS;
        const uint64_t h = vx_blake3_h<NONCE5>(hc, (uint32_t)n, (uint32_t)(n >> 32));
        x ^= (n < count) ? h : 0ull;
    }
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) x ^= __shfl_xor_sync(0xffffffffu, x, d);
    __shared__ uint64_t s[VX_S1_THREADS / 32];
    if ((threadIdx.x & 31) == 0) s[threadIdx.x >> 5] = x;
    __syncthreads();
    if (threadIdx.x == 0) {
        uint64_t y = 0;
        for (int w = 0; w < VX_S1_THREADS / 32; w++) y ^= s[w];
        sink[blockIdx.x] = y;
    }
}

// ----------------------------------------------------------------------------- launches
uint32_t vx_stage1_launches(const VxGeom &g) { return g.wide ? 2u * g.rounds + 3u : 3u; }   // + the clears

cudaError_t vx_launch_stage1(const VxGeom &g, const VxHashConst &hc, uint8_t *ws, cudaStream_t st)
{
    VxCtrl *ctrl = (VxCtrl *)(ws + g.off_ctrl);
    uint32_t *cursor = (uint32_t *)(ws + g.off_cursor);
    // ctrl + cursors (the wide layout's scratch cursors follow the final ones in the workspace plan)
    cudaError_t e = vx_launch_clear(st, ctrl, sizeof(VxCtrl), cursor, g.P * sizeof(uint32_t), nullptr, nullptr);
    if (e != cudaSuccess) return e;
    const uint32_t d_tmp = g.pb - g.pb_tmp;                          // final partitions per scratch partition, log2
    const uint32_t P_tmp = (uint32_t)(g.P >> d_tmp);                 // scratch partitions of this pass
    const uint32_t p_first_tmp = (uint32_t)(g.p_first >> d_tmp);
    if (g.wide) {
        e = vx_launch_clear(st, ws + g.off_cursor_tmp, sizeof(uint32_t) * P_tmp, nullptr, 0, nullptr, nullptr);
        if (e != cudaSuccess) return e;
    }
    const uint64_t per_cta = (uint64_t)VX_S1_THREADS * VX_S1_NPT;
    uint4 *part = (uint4 *)(ws + g.off_part);
    uint16_t *part_b = (uint16_t *)(ws + g.off_part_b);
    if (g.wide) {
        // stage 1 in rounds: hash + one-request scatter of a slice into the scratch partitions
        // (they alias the Table-2 region, unused until stage 2), then compaction into the 10-byte layout
        if (g.pb - g.pb_tmp > 2 || (1u << (g.pb - g.pb_tmp)) > VX_CP_MAXSUB) return cudaErrorInvalidValue;
        uint4 *tmp = (uint4 *)(ws + g.off_tmp);
        uint32_t *cursor_tmp = (uint32_t *)(ws + g.off_cursor_tmp);
        const uint64_t slice = 1ull << g.round_log;
        const uint64_t grid = (slice + per_cta - 1) / per_cta;
        for (uint32_t r = 0; r < g.rounds; r++) {
            if (g.nonce_size == 5)
                vx_k_hash_scatter<true><<<(unsigned)grid, VX_S1_THREADS, 0, st>>>(
                    hc, r * slice, (r + 1) * slice, g.pb_tmp, g.cap_tmp, g.cap_tmp, p_first_tmp, P_tmp, tmp, cursor_tmp, ctrl);
            else
                vx_k_hash_scatter<false><<<(unsigned)grid, VX_S1_THREADS, 0, st>>>(
                    hc, r * slice, (r + 1) * slice, g.pb_tmp, g.cap_tmp, g.cap_tmp, p_first_tmp, P_tmp, tmp, cursor_tmp, ctrl);
            e = cudaGetLastError();
            if (e != cudaSuccess) return e;
            vx_k_compact<<<P_tmp, VX_CP_THREADS, 0, st>>>(
                tmp, cursor_tmp, g.cap_tmp, g.pb, g.pb - g.pb_tmp, g.tile_log, g.cap, g.cap_check,
                (unsigned long long *)part, part_b, cursor, ctrl);
            e = cudaGetLastError();
            if (e != cudaSuccess) return e;
        }
    } else {
        const uint64_t grid = (g.N + per_cta - 1) / per_cta;
        vx_k_hash_scatter<false><<<(unsigned)grid, VX_S1_THREADS, 0, st>>>(hc, 0ull, g.N, g.pb, g.cap, g.cap_check,
                                                                           (uint32_t)g.p_first, (uint32_t)g.P, part, cursor, ctrl);
        e = cudaGetLastError();
        if (e != cudaSuccess) return e;
    }
    vx_k_partition_scan<<<1, VX_SCAN_THREADS, 0, st>>>(cursor, g.cap_check, g.P,
                                                       (unsigned long long *)(ws + g.off_part_base));
    return cudaGetLastError();
}

cudaError_t vx_launch_hash_range(const VxGeom &g, const VxHashConst &hc, uint64_t nonce_begin,
                                 uint64_t count, uint64_t *dev_hashes, cudaStream_t st)
{
    if (count == 0) return cudaSuccess;
    const uint64_t grid = (count + VX_S1_THREADS - 1) / VX_S1_THREADS;
    if (g.nonce_size == 5)
        vx_k_hash_range<true><<<(unsigned)grid, VX_S1_THREADS, 0, st>>>(hc, nonce_begin, count, dev_hashes);
    else
        vx_k_hash_range<false><<<(unsigned)grid, VX_S1_THREADS, 0, st>>>(hc, nonce_begin, count, dev_hashes);
    return cudaGetLastError();
}

cudaError_t vx_launch_hash_sink(const VxGeom &g, const VxHashConst &hc, uint64_t count,
                                uint64_t *dev_sink, size_t sink_words, cudaStream_t st)
{
    const uint64_t per_cta = (uint64_t)VX_S1_THREADS * VX_S1_NPT;
    const uint64_t grid = (count + per_cta - 1) / per_cta;
    if (grid == 0) return cudaSuccess;
    if (grid > sink_words) return cudaErrorInvalidValue;
    if (g.nonce_size == 5)
        vx_k_hash_sink<true><<<(unsigned)grid, VX_S1_THREADS, 0, st>>>(hc, count, dev_sink);
    else
        vx_k_hash_sink<false><<<(unsigned)grid, VX_S1_THREADS, 0, st>>>(hc, count, dev_sink);
    return cudaGetLastError();
}

// ----------------------------------------------------------------------------- Table-2 re-keying (8(f2))
// SURVEY.md 8(f2) / PAPER.md L49, L65, L77: a prover looks a challenge up by hash, but Table 2 leaves
// the match step grouped by the bucket of the TABLE-1 hash.  Readings A19/A20: every pair
// is hashed, H2 = BLAKE3 keyed hash of nonce1 || nonce2 (the same compression as stage 1 with message
// words m0 = n1, m1 = n2 and block_len 8), and the pairs are bucketed by H2 exactly as stage 1 buckets
// nonces: atomic append of {H2, index of the pair in Table 2} into the coarse hash-prefix partitions
// -- the partition array of Table 1, which has done its job -- then the fused kernel sorts every
// partition (no matching) and writes the CSR offsets.  The pairs themselves stay where they are; the
// export gathers them in H2 order.
__global__ void __launch_bounds__(VX_S1_THREADS)
vx_k_rekey_scatter(const __grid_constant__ VxHashConst hc2, const uint2 *__restrict__ t2_rec, uint32_t pb,
                   uint32_t cap, uint32_t cap_check, uint4 *__restrict__ part, uint32_t *__restrict__ cursor,
                   VxCtrl *__restrict__ ctrl)
{
    const unsigned long long M = ctrl->t2_total;
    const uint64_t base = (uint64_t)blockIdx.x * (VX_S1_THREADS * VX_S1_NPT) + threadIdx.x;
    if ((uint64_t)blockIdx.x * (VX_S1_THREADS * VX_S1_NPT) >= M) return;
    if (M > 0xffffffffull) {                            // the pair index is kept in 32 bits
        if (base == 0) atomicOr(&ctrl->flags, VX_FLAG_T2_OVERFLOW);
        return;
    }
    uint64_t H[VX_S1_NPT];
#pragma unroll
    for (int k = 0; k < VX_S1_NPT; k++) {
        const uint64_t r = base + (uint64_t)k * VX_S1_THREADS;
        const uint2 pr = r < M ? __ldcs(t2_rec + r) : make_uint2(0u, 0u);
        H[k] = vx_blake3_h<true>(hc2, pr.x, pr.y);
    }
#pragma unroll
    for (int k = 0; k < VX_S1_NPT; k++) {
        const uint64_t r = base + (uint64_t)k * VX_S1_THREADS;
        if (r < M) {
            const uint32_t p = pb ? (uint32_t)(H[k] >> (64 - pb)) : 0u;
            const uint32_t slot = atomicAdd(&cursor[p], 1u);
            if (slot < cap_check)
                part[(uint64_t)p * cap + slot] = make_uint4((uint32_t)H[k], (uint32_t)(H[k] >> 32), (uint32_t)r, 0u);
            else
                atomicOr(&ctrl->flags, VX_FLAG_PART_OVERFLOW);
        }
    }
}

// the Table-1 record count, kept for vx_get_stats before the partition bases are rebuilt for the pairs
__global__ void vx_k_save_t1_total(const unsigned long long *__restrict__ part_base, uint64_t P, VxCtrl *__restrict__ ctrl)
{
    ctrl->t1_total = part_base[P];
}

// The same in the wide layout (K >= 33, or forced): Table 2 is resident packed (uint2 {n1 lo, n2 lo} + a
// byte of high bits) and the partition array holds 10-byte records -- a = (H2 << pb) | (index >> 16),
// b = index & 0xffff: the pb bits the prefix frees hold the high bits of the 33-bit pair index, exactly as
// they hold the high nonce bits in Table 1, so the wide sort kernel orders (a, b) = (H2, index) unchanged.
// Two scattered stores per record (the scratch of stage 1's rounds aliases the Table-2 region, which is
// live here): 1.8x the one-store kernel, off the plot path.
template <bool NONCE5>
__global__ void __launch_bounds__(VX_S1_THREADS)
vx_k_rekey_scatter_wide(const __grid_constant__ VxHashConst hc2, const uint2 *__restrict__ t2_rec,
                        const uint8_t *__restrict__ t2_hi, uint32_t pb, uint32_t cap, uint32_t cap_check,
                        unsigned long long *__restrict__ part_a, uint16_t *__restrict__ part_b,
                        uint32_t *__restrict__ cursor, VxCtrl *__restrict__ ctrl)
{
    const unsigned long long M = ctrl->t2_total;
    const uint64_t base = (uint64_t)blockIdx.x * (VX_S1_THREADS * VX_S1_NPT) + threadIdx.x;
    if ((uint64_t)blockIdx.x * (VX_S1_THREADS * VX_S1_NPT) >= M) return;
    if (pb + 16 < 64 && (M >> (pb + 16)) != 0) {        // the pair index must fit pb + 16 bits
        if (base == 0) atomicOr(&ctrl->flags, VX_FLAG_T2_OVERFLOW);
        return;
    }
    uint64_t H[VX_S1_NPT];
#pragma unroll
    for (int k = 0; k < VX_S1_NPT; k++) {
        const uint64_t r = base + (uint64_t)k * VX_S1_THREADS;
        const uint2 pr = r < M ? __ldcs(t2_rec + r) : make_uint2(0u, 0u);
        if constexpr (NONCE5) {
            const uint32_t hb = r < M ? t2_hi[r] : 0u;  // (n1 >> 32) | (n2 >> 32) << 4
            // message bytes: n1[0..4] n2[0..4]
            const uint32_t m1 = (hb & 15u) | (pr.y << 8);
            const uint32_t m2 = (pr.y >> 24) | ((hb >> 4) << 8);
            H[k] = vx_blake3_h3(hc2, pr.x, m1, m2);
        } else {
            H[k] = vx_blake3_h<true>(hc2, pr.x, pr.y);
        }
    }
#pragma unroll
    for (int k = 0; k < VX_S1_NPT; k++) {
        const uint64_t r = base + (uint64_t)k * VX_S1_THREADS;
        if (r < M) {
            const uint32_t p = pb ? (uint32_t)(H[k] >> (64 - pb)) : 0u;
            const uint32_t slot = atomicAdd(&cursor[p], 1u);
            if (slot < cap_check) {
                const size_t at = (size_t)p * cap + slot;
                part_a[at] = (pb ? H[k] << pb : H[k]) | (r >> 16);
                part_b[at] = (uint16_t)(r & 0xffffu);
            } else {
                atomicOr(&ctrl->flags, VX_FLAG_PART_OVERFLOW);
            }
        }
    }
}

cudaError_t vx_launch_rekey(const VxGeom &g, const VxHashConst &hc2, uint8_t *ws, cudaStream_t st)
{
    if (g.passes_log) return cudaErrorInvalidValue;
    VxCtrl *ctrl = (VxCtrl *)(ws + g.off_ctrl);
    uint32_t *cursor = (uint32_t *)(ws + g.off_cursor);
    vx_k_save_t1_total<<<1, 1, 0, st>>>((const unsigned long long *)(ws + g.off_part_base), g.P, ctrl);
    cudaError_t e = cudaGetLastError();
    if (e == cudaSuccess) e = vx_launch_clear(st, cursor, g.P * sizeof(uint32_t), nullptr, 0, nullptr, nullptr);
    if (e != cudaSuccess) return e;
    const uint64_t per_cta = (uint64_t)VX_S1_THREADS * VX_S1_NPT;
    const uint64_t grid = (g.t2_cap + per_cta - 1) / per_cta;          // upper bound; CTAs beyond |Table 2| exit
    if (g.wide) {
        unsigned long long *part_a = (unsigned long long *)(ws + g.off_part);
        uint16_t *part_b = (uint16_t *)(ws + g.off_part_b);
        if (g.nonce_size == 5)
            vx_k_rekey_scatter_wide<true><<<(unsigned)grid, VX_S1_THREADS, 0, st>>>(
                hc2, (const uint2 *)(ws + g.off_t2_rec), ws + g.off_t2_hi, g.pb, g.cap, g.cap_check, part_a, part_b, cursor, ctrl);
        else
            vx_k_rekey_scatter_wide<false><<<(unsigned)grid, VX_S1_THREADS, 0, st>>>(
                hc2, (const uint2 *)(ws + g.off_t2_rec), ws + g.off_t2_hi, g.pb, g.cap, g.cap_check, part_a, part_b, cursor, ctrl);
    } else {
        vx_k_rekey_scatter<<<(unsigned)grid, VX_S1_THREADS, 0, st>>>(hc2, (const uint2 *)(ws + g.off_t2_rec), g.pb, g.cap,
                                                                     g.cap_check, (uint4 *)(ws + g.off_part), cursor, ctrl);
    }
    e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    vx_k_partition_scan<<<1, VX_SCAN_THREADS, 0, st>>>(cursor, g.cap_check, g.P,
                                                       (unsigned long long *)(ws + g.off_part_base));
    return cudaGetLastError();
}

// ----------------------------------------------------------------------------- one plot over G GPUs: launches
cudaError_t vx_launch_shard_clear(const VxGeom &g, uint8_t *ws, cudaStream_t st)
{
    return vx_launch_clear(st, ws + g.off_ctrl, sizeof(VxCtrl), ws + g.off_cursor, g.P * sizeof(uint32_t), nullptr, nullptr);
}

cudaError_t vx_launch_shard_scatter(const VxGeom &g, const VxHashConst &hc, uint32_t rank, uint32_t world_log,
                                    uint8_t *const *peer_ws, cudaStream_t st)
{
    if (g.wide || world_log != g.passes_log || world_log == 0 || (1u << world_log) > VX_MAX_SHARD_WORLD)
        return cudaErrorInvalidValue;
    VxPeers peers;
    for (uint32_t i = 0; i < VX_MAX_SHARD_WORLD; i++) peers.ws[i] = i < (1u << world_log) ? peer_ws[i] : nullptr;
    const uint64_t share = g.N >> world_log, n0 = (uint64_t)rank * share;
    const uint64_t per_cta = (uint64_t)VX_S1_THREADS * VX_S1_NPT;
    const uint64_t grid = (share + per_cta - 1) / per_cta;
    vx_k_hash_scatter_sharded<<<(unsigned)grid, VX_S1_THREADS, 0, st>>>(hc, peers, n0, n0 + share, g.pb,
                                                                        g.pb - world_log, g.cap, g.cap_check,
                                                                        g.off_part, g.off_cursor, g.off_ctrl);
    return cudaGetLastError();
}

cudaError_t vx_launch_shard_scan(const VxGeom &g, uint8_t *ws, cudaStream_t st)
{
    vx_k_partition_scan<<<1, VX_SCAN_THREADS, 0, st>>>((const uint32_t *)(ws + g.off_cursor), g.cap_check, g.P,
                                                       (unsigned long long *)(ws + g.off_part_base));
    return cudaGetLastError();
}

