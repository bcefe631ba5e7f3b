// vx_internal.h -- geometry, workspace plan and launch wrappers shared by the .cu files of libvx.
// Not part of the public ABI (that is include/vx.h).
#pragma once
#include <cuda_runtime.h>
#include <stddef.h>
#include <stdint.h>

#include "vx_blake3.cuh"

// ---------------------------------------------------------------------------------- geometry
// Hierarchical bucketing: stage 1 scatters records into 2^pb coarse
// hash-prefix partitions of ~2^VX_TILE_LOG records each (they fit one CTA's shared memory);
// stage 2 splits a partition into its 2^fb buckets (fb = B - pb) with a shared-memory
// distribution sort over VX_BIN_BITS more hash bits (about one record per bin).
#define VX_TILE_LOG 12          // log2 of the mean records per partition, K <= 31
#define VX_S2_THREADS 512
#define VX_S2_ITEMS 9           // VX_S2_THREADS * VX_S2_ITEMS >= partition capacity (mean + 8 sigma)
#define VX_S2_MINB 2            // resident CTAs per SM the fused kernel is compiled for
// K >= 32: 2^(K-12) open partitions no longer stay resident in L2 during stage 1 (K=32 stage 1 was
// 139 ms instead of 2 x 54); tiles of 2^13 records halve their number.  One 1024-thread CTA per SM.
#define VX_TILE_LOG_BIG 13
#define VX_S2B_THREADS 1024
#define VX_S2B_ITEMS 9
#define VX_BIG_TILES_FROM_K 32
#define VX_STAGE_MAX_BYTES ((size_t)64 << 20) // Table-1 export staging (vx_read_tables)
#define VX_MAX_MEAN_BUCKET_LOG 9 // K - B - passes_log <= 9: at most 2^33 records resident (BASELINE.json K=33)
#define VX_MAX_K 36              // wide Table-2 records keep 4 high nonce bits per nonce
#define VX_MAX_PASSES_LOG 8

struct VxGeom {
    uint32_t K, B, nonce_size;
    uint32_t wide; // compact 10-byte internal Table-1 records + 9-byte Table-2 records (K >= 33, or forced)
    uint32_t tile_log; // log2 of the mean partition size: VX_TILE_LOG or VX_TILE_LOG_BIG
    uint32_t pb;   // partition bits: partition = H >> (64 - pb)
    uint32_t fb;   // bucket bits inside a partition, B - pb
    uint32_t cap;  // partition capacity in records (mean + slack, multiple of 32)
    uint32_t cap_check;   // = cap; a test hook lowers it (the slot stride stays cap) to raise the overflow error
    uint64_t t2_check;    // = t2_cap; likewise for Table 2
    uint32_t subkey_bits; // = 32: hash bits below the bin index that stage 2's fast ranking compares; a test hook
                          // narrows it so that the tie -> exact re-rank path of a tile runs under test
    uint32_t s2_kernel;   // 0: the classic fused kernel; 1: the warp-local variant where it applies (VX_OPT_STAGE2_KERNEL)
    uint64_t N;    // 2^K
    uint64_t P;    // partitions resident at a time: 2^(pb - passes_log)
    uint64_t NB;   // 2^B
    // Bucket-range passes: the plot is made in 2^passes_log passes;
    // pass s hashes ALL 2^K nonces but keeps only the records whose top passes_log hash bits are s,
    // i.e. the partitions [p_first, p_first + P) and the buckets [b_first, b_first + NBp).  The
    // workspace holds one pass; partition, tile and offset indices inside the kernels are relative
    // to the pass (pb stays the global partition-bit count: it is part of the wide key format).
    uint32_t passes_log, pass;
    uint64_t p_first, b_first, NBp;
    uint64_t t2_cap; // Table-2 capacity in records
    uint32_t rec1_bytes, rec2_bytes;
    // workspace carve-up (byte offsets, each 256-aligned)
    size_t off_ctrl, off_cursor, off_part_base, off_status;
    size_t off_part;   // partition records: uint4 {H lo, H hi, nonce lo, nonce hi} per record;
                       // after stage 2 each partition is sorted: this IS the resident Table 1.
                       // wide: uint64 a = (H << pb) | (n >> tile_log) per record (the partition prefix of H is
                       // implied, the freed pb bits hold the high nonce bits) ...
    size_t off_part_b; // ... wide only: uint16 b = n & (2^tile_log - 1) per record (same slot numbering)
    size_t off_t1_off, off_t2_off, off_t2_rec;
    size_t off_t2_hi;  // wide only: uint8 per Table-2 record, (n1 >> 32) | (n2 >> 32) << 4
    size_t off_stage, stage_bytes;   // export staging for vx_read_tables(Table 1)
    // wide only -- stage 1 in rounds: the nonce space is hashed in
    // `rounds` slices of 2^round_log nonces; each slice is scattered as 16-byte records (one store
    // request per record) into 2^pb_tmp coarse partitions of a scratch area that aliases the not yet
    // used Table-2 region, then compacted into the 10-byte partition array with coalesced stores.
    uint32_t rounds, round_log, pb_tmp, cap_tmp;
    size_t off_cursor_tmp, off_tmp;
    size_t total;
};

// device-resident control block (first bytes of the workspace)
struct VxCtrl {
    uint32_t ticket;      // stage-2 tile dispenser
    uint32_t flags;       // bit 0: partition slack overflow, bit 1: Table-2 capacity overflow
    uint32_t max_bucket;  // largest Table-1 bucket seen by stage 2
    uint32_t retries;     // tiles that stage 2 re-ranked exactly after its fast ranking met a tie
    unsigned long long t2_total;  // number of Table-2 records
    unsigned long long t1_total;  // Table-1 records, saved by vx_rekey_table2 before the partition bases are rebuilt
};
#define VX_FLAG_PART_OVERFLOW 1u
#define VX_FLAG_T2_OVERFLOW 2u
#define VX_FLAG_BOUNDS 4u        // a VX_CHECK failed (debug build only)
// Index checks of our own (compute-sanitizer is not available on the GPU pool): built with
// -DVX_DEBUG_BOUNDS=1 (VX_NVCC_EXTRA, paper_2606_14007_b200/build.py) every shared- and global-memory
// index of the kernels is checked against its array and a failure surfaces as VX_ERR_CUDA
// "internal bounds check failed" at the next synchronising call.  Empty in the product build.
#ifndef VX_DEBUG_BOUNDS
#define VX_DEBUG_BOUNDS 0
#endif
#if VX_DEBUG_BOUNDS
#define VX_CHECK(ctrl, cond) do { if (!(cond)) atomicOr(&(ctrl)->flags, VX_FLAG_BOUNDS); } while (0)
#else
#define VX_CHECK(ctrl, cond) do { } while (0)
#endif

// accessors of the opaque handle (vx_api.cu) for the other .cu files: its folded hash constants, and its
// error text set the way every ABI call sets it
struct vx_plot;
const VxHashConst &vx_plot_hash_const(const vx_plot *p);
int vx_plot_fail(vx_plot *p, int status, const char *what);                 // returns status (a vx_status)
int vx_plot_fail_cuda(vx_plot *p, cudaError_t e, const char *what);         // returns VX_ERR_CUDA
// returns false if (K, B) is not a supported geometry
bool vx_geom_init(VxGeom *g, uint32_t K, uint32_t B, bool force_wide, bool force_big_tiles, uint32_t passes_log = 0);
void vx_geom_select_pass(VxGeom *g, uint32_t pass);

// host fold of the nonce-independent part of round 1 (vx_blake3.cuh)
void vx_hash_const_init(VxHashConst *hc, const uint8_t key[32], uint32_t nonce_size);

// ---------------------------------------------------------------------------------- launches
cudaError_t vx_launch_stage1(const VxGeom &g, const VxHashConst &hc, uint8_t *ws, cudaStream_t st);
uint32_t vx_stage1_launches(const VxGeom &g);   // kernels vx_launch_stage1 enqueues
// one plot over G = 2^world_log GPUs (8(f4)): clear the rank's cursors; hash the rank's nonce share and
// scatter every record into its owner's workspace (peer_ws[g] = base of rank g's workspace, device
// pointers valid on this device); scan the rank's own partitions.  The caller puts a barrier over all
// ranks between the three.
#define VX_MAX_SHARD_WORLD 8
cudaError_t vx_launch_shard_clear(const VxGeom &g, uint8_t *ws, cudaStream_t st);
cudaError_t vx_launch_shard_scatter(const VxGeom &g, const VxHashConst &hc, uint32_t rank, uint32_t world_log,
                                    uint8_t *const *peer_ws, cudaStream_t st);
cudaError_t vx_launch_shard_scan(const VxGeom &g, uint8_t *ws, cudaStream_t st);
// Table-2 re-keying (8(f2)): hash every pair (hc2: block_len = 2 NONCE_SIZE), append {H2, pair index}
// to the hash-prefix partitions (the partition array of Table 1 is reused), scan.  Then
// vx_launch_stage2(do_match = false) sorts the partitions and writes the CSR offsets.
cudaError_t vx_launch_rekey(const VxGeom &g, const VxHashConst &hc2, uint8_t *ws, cudaStream_t st);
// re-keyed pairs [first, first + count) of the CSR numbering, gathered through the sorted pair indices
// into the external Table-2 format in ws + off_stage
cudaError_t vx_launch_export_rekey(const VxGeom &g, uint8_t *ws, uint64_t first, uint64_t count, cudaStream_t st);
// zero two regions and two words with a kernel (not a memset: see vx_k_clear)
cudaError_t vx_launch_clear(cudaStream_t st, void *a, size_t bytes_a, void *b, size_t bytes_b, uint32_t *w0, uint32_t *w1);
// sorts (and matches) the partitions [tile_begin, tile_end) -- (0, P) for the whole plot; slices must
// be launched in ascending order on one stream.  slice_end_out (host-mapped, may be NULL) receives
// the number of Table-2 records of the partitions < tile_end.
cudaError_t vx_launch_stage2(const VxGeom &g, uint8_t *ws, bool do_match, bool force_exact, int num_sms,
                             cudaStream_t st, uint32_t tile_begin = 0, uint32_t tile_end = 0xffffffffu,
                             unsigned long long *slice_end_out = nullptr);
// external-format Table-1 records [first, first + count) of the CSR numbering -> ws + off_stage
cudaError_t vx_launch_export_t1(const VxGeom &g, uint8_t *ws, uint64_t first, uint64_t count, cudaStream_t st);
// wide, NONCE_SIZE = 5: external 10-byte Table-2 records [first, first + count) -> ws + off_stage
cudaError_t vx_launch_export_t2(const VxGeom &g, uint8_t *ws, uint64_t first, uint64_t count, cudaStream_t st,
                                size_t stage_offset = 0);   // ... + stage_offset
cudaError_t vx_launch_hash_range(const VxGeom &g, const VxHashConst &hc, uint64_t nonce_begin,
                                 uint64_t count, uint64_t *dev_hashes, cudaStream_t st);
cudaError_t vx_launch_hash_sink(const VxGeom &g, const VxHashConst &hc, uint64_t count,
                                uint64_t *dev_sink, size_t sink_words, cudaStream_t st);
// Table-2 egress (vx_egress.cu): stage 2 in `slices` partition-range launches on `compute`, each
// finished slice copied on `copy` to host memory (host_records / host_offsets) or, through a pinned
// ring of 4 MB chunks, to a file.  *soft_error: 0 ok, 1 capacity too small, 2 Table-2 overflow, 3 I/O,
// 4 too many egress calls in flight.
int vx_write_all(int fd, const uint8_t *src, size_t bytes, uint64_t *written, char *err, size_t errlen);
int vx_sm_count(void);   // SMs of the current device (cached per ordinal); 148 if the query fails
struct VxRing;
VxRing *vx_ring_create(void *pinned, size_t bytes, int fd);   // NULL: fewer than two 4 MB chunks, or no memory
uint64_t vx_ring_written(const VxRing *r);
void vx_ring_destroy(VxRing *r);
cudaError_t vx_egress_run(const VxGeom &g, uint8_t *ws, bool force_exact, int num_sms, cudaStream_t compute,
                          cudaStream_t copy, uint32_t slices, uint8_t *host_records, size_t records_capacity,
                          uint64_t *host_offsets, VxRing *ring, uint64_t *t2_records, VxCtrl *ctrl_out,
                          int *soft_error, char *err, size_t errlen);
cudaError_t vx_stage2_configure(void); // opt in to the large dynamic shared memory once
size_t vx_stage2_smem_bytes(const VxGeom &g);
