/*
 * vx.h -- C ABI of the B200-native VaultxGPU plotting hot path (libvx.so).
 *
 * The library computes, for a plot (K, key):
 *
 *   Table 1  all 2^K records (n, H(n)), n in [0, 2^K), H(n) = first 8 bytes of the BLAKE3 keyed
 *            hash of the NONCE_SIZE little-endian bytes of n (read big-endian), grouped into 2^24
 *            buckets by the hash prefix  H >> 40       (PAPER.md L41-43 I-A, L81 III-A, L91 III-B)
 *   Table 2  for every bucket, every pair of its records whose hashes differ by less than
 *            T = 2^(64-K), as (n_first, n_second), first = smaller (H, n)
 *                                                       (PAPER.md L65 II-B, L81 III-A)
 *
 * PAPER.md = /root/reference/PAPER.md (arxiv/paper_2606_14007).  Where the paper leaves the record
 * layout, widths, bucket rule or predicate open, the readings are A1..A18 of SURVEY.md 8(c),
 * restated in DESIGN.md.  Everything runs in hand-written CUDA kernels for sm_100a; there is no
 * CPU fallback: without a CUDA device every compute call returns VX_ERR_CUDA.
 *
 * Conventions
 *   - every call returns vx_status (no exceptions, no errno, no abort);
 *   - `dev_*` pointers are DEVICE pointers owned by the caller (PyTorch), `host` pointers are
 *     ordinary or pinned host memory owned by the caller; the library allocates no device memory
 *     of its own and never frees the caller's;
 *   - `cuda_stream` is a cudaStream_t passed as void* (NULL = the legacy default stream);
 *   - vx_build_table1 / vx_sort_match_table2 only ENQUEUE work on that stream and return; errors
 *     raised on the device (slack overflow) surface as VX_ERR_OVERFLOW at the next synchronising
 *     call (vx_read_tables, vx_get_stats, vx_synchronize);
 *   - handles are independent: the key travels as a kernel parameter (constant bank), not in a
 *     module-global __constant__, so plots with different keys can coexist.
 *
 * External record formats (reading A1, A4, A12; SURVEY.md 8(c) Step 5)
 *   NONCE_SIZE = 4 for K <= 32, 5 for 33 <= K <= 40
 *   Table-1 record: nonce[NONCE_SIZE] little-endian || hash[8]  (the 8 digest bytes, = H big-endian)
 *   Table-2 record: nonce1[NONCE_SIZE] || nonce2[NONCE_SIZE], little-endian
 *   offsets: uint64, CSR style, (number of buckets + 1) entries, in records.
 */
#ifndef VX_H_
#define VX_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct vx_plot vx_plot; /* opaque; owns only host metadata */

typedef enum {
    VX_OK = 0,
    VX_ERR_ARG = -1,       /* bad argument (NULL, K out of range, bucket range reversed ...)      */
    VX_ERR_STATE = -2,     /* call out of order (e.g. sort_match before build, read before bind)  */
    VX_ERR_WORKSPACE = -3, /* bound workspace smaller than vx_workspace_bytes / misaligned        */
    VX_ERR_CUDA = -4,      /* a CUDA runtime call failed; text in vx_last_error                    */
    VX_ERR_OVERFLOW = -5,  /* a partition's slack or the Table-2 capacity overflowed on the device */
    VX_ERR_RANGE = -6,     /* bucket range outside [0, 2^B] or records_capacity too small          */
    VX_ERR_UNSUPPORTED = -7, /* a valid request beyond a fixed limit of this build (e.g. more than 16
                                Table-2 egress calls in flight in one process); text in vx_last_error   */
    VX_ERR_IO = -8,         /* write() to the egress file descriptor failed; text in vx_last_error    */
    VX_ERR_NOMEM = -9       /* host memory for the handle could not be allocated                      */
} vx_status;

/* Device bytes the caller must provide for a plot of this K (B = 24 buckets bits, the paper's
 * setting).  0 if K is out of range.  Host-only arithmetic, no CUDA call. */
size_t vx_workspace_bytes(uint32_t K);
/* Same for a test-only bucket_bits (see vx_plot_create_ex). */
size_t vx_workspace_bytes_ex(uint32_t K, uint32_t bucket_bits);

/* Create a plot handle for 2^K nonces under a 256-bit key (host pointer, copied).  K in 1..36 with
 * 2^24 buckets; K >= 33 uses 5-byte nonces (reading A1) and the compact "wide" internal layout
 * below.  Up to K = 33 (BASELINE.json's largest configuration, mean bucket 512 records, 171 GB) the
 * whole plot is resident at once; K = 34..36 is made in 2^(K-33) bucket-range PASSES (below), each
 * the size of a K = 33 plot.  (SURVEY.md 8(b) allowed K up to 40: beyond 36 the packed Table-2 record
 * of the wide layout, 4 high nonce bits per nonce, would have to grow.)  PAPER.md L41-43. */
vx_status vx_plot_create(uint32_t K, const uint8_t key[32], vx_plot **out);
/* Test-only: bucket_bits B in 1..24 instead of 24 (dense buckets at tiny K, reading A7). */
vx_status vx_plot_create_ex(uint32_t K, const uint8_t key[32], uint32_t bucket_bits, vx_plot **out);
/* Test-only flags.  VX_CREATE_WIDE_LAYOUT: use the K >= 33 internal layout at this K, so that the
 * wide kernels can be compared with the oracle on full small tables (results are identical by
 * construction; the external formats do not change). */
#define VX_CREATE_WIDE_LAYOUT 1u
/* VX_CREATE_BIG_TILES: use the K >= 32 tile geometry (2^13-record partitions, one 1024-thread CTA
 * per SM) at this K, for the same reason. */
#define VX_CREATE_BIG_TILES 2u
/* VX_CREATE_PASSES_LOG(l): make the plot in 2^l bucket-range passes (l in 1..8; l <= partition bits)
 * whatever K is -- the test-only "VRAM budget" with which the multi-pass path is compared with the
 * oracle on small tables.  Without it K <= 33 takes one pass and K >= 34 the fewest that fit. */
#define VX_CREATE_PASSES_LOG_SHIFT 8
#define VX_CREATE_PASSES_LOG_MASK 0xf00u
#define VX_CREATE_PASSES_LOG(l) ((uint32_t)(l) << VX_CREATE_PASSES_LOG_SHIFT)
vx_status vx_plot_create_opts(uint32_t K, const uint8_t key[32], uint32_t bucket_bits, uint32_t flags,
                              vx_plot **out);
size_t vx_workspace_bytes_opts(uint32_t K, uint32_t bucket_bits, uint32_t flags);

/* Attach caller-owned device memory (>= vx_workspace_bytes, 256-byte aligned).  The workspace
 * holds Table 1 (the partition array), Table 2, their offsets, the look-back state and a small
 * export staging area for the life of the plot. */
vx_status vx_plot_bind(vx_plot *p, void *dev_workspace, size_t bytes);

/* Stage 1: hash every nonce and place its record
 * into its hash-prefix partition in HBM.  Enqueues only.  After it, Table 1 is resident in HBM as
 * 2^P coarse hash-prefix buckets (P = max(K-12, 0) capped at B); the split of each coarse bucket
 * into its 2^(B-P) buckets is an in-shared-memory counting step of the fused kernel below (or
 * of vx_read_tables when Table 1 is read before vx_sort_match_table2).  See DESIGN.md "hierarchy".
 * Wide layout (K >= 33): the nonce space is hashed in 4 rounds; each round scatters its records,
 * 16 bytes each, into scratch partitions that alias the (still unused) Table-2 region and then
 * compacts them into the 10-byte partition array. */
vx_status vx_build_table1(vx_plot *p, void *cuda_stream);

/* Stage 2 (rows a6-a8; "fused ... single GPU kernel"): for every bucket, stage it in
 * shared memory, sort by (H, n), apply the match predicate, write the sorted bucket back to
 * Table 1 in place (reading A14) and the matches to Table 2, with exact CSR offsets for both.
 * Enqueues only. */
vx_status vx_sort_match_table2(vx_plot *p, void *cuda_stream);

/* Table-2 egress pipeline ("transferred from VRAM to host over PCIe and
 * written to disk in 4 MB sequential chunks", L91 pinned staging buffer, L165/L169 "overlap the PCIe
 * transfer with GPU computation using async streams").  Both calls replace vx_sort_match_table2: the
 * fused sort + match stage runs as `slices` launches over consecutive partition ranges on
 * compute_stream (1..256; clamped), and the Table-2 records and CSR offsets of each finished slice
 * are copied on copy_stream (a different stream) while the later slices are still being matched.
 * Both BLOCK until everything has arrived and report device-raised errors like vx_synchronize.
 * With 5-byte nonces (K = 33) Table 2 is resident in a packed form: each chunk is first converted to
 * the external format in the workspace's staging area (a kernel on copy_stream), then copied.
 *
 * _to_host: host_records (HOST, caller-owned, pinned for the copies to overlap; records_capacity
 *   bytes, VX_ERR_RANGE if too small) receives all of Table 2 in the external format, bucket-major;
 *   host_offsets (HOST, 2^B + 1 entries, may be NULL) the CSR offsets; *records_bytes the size.
 * _to_file: the same stream of bytes goes to file descriptor fd with sequential write()s of 4 MB
 *   through pinned_staging (HOST, pinned, caller-owned, >= 8 MB; used as a ring of 4 MB chunks, up
 *   to 1024 of them): records, then the (2^B + 1) uint64 offsets, then a 32-byte trailer
 *   {"VXT2\0\0\0\1", u32 K, u32 B, u32 NONCE_SIZE, u32 pass | log2(passes) << 16, u64 |Table 2|}
 *   (a plot made in passes, below: the records and the 2^B / passes + 1 offsets of the selected pass).  The paper's plot-file
 *   format is unpublished; this layout is this library's own.  *file_bytes = bytes
 *   written.  VX_ERR_IO if a write fails. */
vx_status vx_sort_match_table2_to_host(vx_plot *p, void *compute_stream, void *copy_stream, uint32_t slices,
                                       void *host_records, size_t records_capacity, uint64_t *host_offsets,
                                       size_t *records_bytes);
vx_status vx_sort_match_table2_to_file(vx_plot *p, void *compute_stream, void *copy_stream, uint32_t slices,
                                       int fd, void *pinned_staging, size_t staging_bytes, uint64_t *file_bytes);

/* Table-2 re-keying and the plot file (PAPER.md L49 / L77 "plot files ... searched by
 * the ... prover", L65 the four-stage pipeline ending in the file).  Table 2 leaves the match step
 * grouped by the bucket of the Table-1 hash; a prover looks a challenge up by the hash of the PAIR.
 * The paper gives neither that hash nor the file layout and VaultX is unpublished (L183): readings
 * A19-A21 of DESIGN.md are this library's own (parity with VaultX unpinned).
 *   vx_rekey_table2   after vx_sort_match_table2*: hash every pair, H2 = first 8 bytes (big-endian) of
 *                     the BLAKE3 keyed hash of nonce1 LE || nonce2 LE under the plot key, and bucket
 *                     the pairs by H2 >> (64 - B), each bucket in H2 order, with CSR offsets.  The
 *                     {H2, pair index} records are built in Table 1's partition array: TABLE 1 IS GONE
 *                     afterwards (vx_read_tables(1) / vx_device_tables return VX_ERR_STATE), Table 2
 *                     itself stays readable.  Enqueues only.  One-pass plots (K <= 33; with 5-byte
 *                     nonces the 10 message bytes are three BLAKE3 message words and the records are
 *                     kept in the wide 10-byte layout, a = (H2 << pb) | (index >> 16), b = index &
 *                     0xffff); a plot made in passes returns VX_ERR_UNSUPPORTED (the pair hash scatters
 *                     over all buckets: every pair must be resident).
 *   vx_read_tables(p, VX_TABLE2_REKEYED, ...)  the re-keyed buckets in the external Table-2 record
 *                     format (the order of pairs with equal H2 is unspecified, reading A20).
 *   vx_write_plot_file  header "VXPLOT\0\1" | u32 K | u32 B | u32 NONCE_SIZE | u32 0 | key[32] |
 *                     u64 records, then the 2^B + 1 u64 offsets, then the records bucket-major, all
 *                     little-endian, written to fd with sequential write()s through pinned_staging
 *                     (HOST, >= 1 MB).  Blocks.  *file_bytes = bytes written. */
#define VX_TABLE2_REKEYED 3
vx_status vx_rekey_table2(vx_plot *p, void *cuda_stream);
vx_status vx_write_plot_file(vx_plot *p, int fd, void *pinned_staging, size_t staging_bytes, uint64_t *file_bytes);

/* Bucket-range passes (VI: "chunked VRAM tiling to handle k > 31
 * without requiring the full Table-1 in VRAM").  A plot with P = 2^l passes is made one hash-prefix
 * slice at a time: pass s hashes ALL 2^K nonces but keeps only the records whose top l hash bits are
 * s, i.e. the buckets [s 2^B / P, (s + 1) 2^B / P); Table 1, Table 2 and their offsets of that slice
 * occupy the workspace (sized for one pass) until the next pass is selected.  The buckets of
 * different passes are disjoint and complete, so the passes together are exactly the one-pass plot.
 *   vx_plot_passes       P, the selected pass and its bucket range (any pointer may be NULL);
 *   vx_plot_select_pass  choose the slice that vx_build_table1 / vx_sort_match_table2* / vx_read_tables
 *                        / vx_get_stats act on (default 0; reads outside its bucket range return
 *                        VX_ERR_RANGE; vx_get_stats counts the slice).  Synchronises; the previous
 *                        slice's tables are gone afterwards;
 *   vx_plot_all_passes_to_host  the whole plot: for every pass, vx_build_table1 and the streamed egress
 *                        of vx_sort_match_table2_to_host, Table 2 appended to host_records (HOST,
 *                        records_capacity bytes) and the CSR offsets of all 2^B buckets (global, in
 *                        records) written to host_offsets (HOST, 2^B + 1 entries, may be NULL).
 *                        *records_bytes = bytes written, *t1_records = records placed over all passes
 *                        (= 2^K).  Blocks.  One pass: the same as build + _to_host. */
vx_status vx_plot_passes(const vx_plot *p, uint32_t *passes, uint32_t *selected, uint64_t *bucket_begin,
                         uint64_t *bucket_end);
vx_status vx_plot_select_pass(vx_plot *p, uint32_t pass);
vx_status vx_plot_all_passes_to_host(vx_plot *p, void *compute_stream, void *copy_stream, uint32_t slices,
                                     void *host_records, size_t records_capacity, uint64_t *host_offsets,
                                     size_t *records_bytes, uint64_t *t1_records);

/* One plot over G = 2, 4 or 8 GPUs (the paper's machines hold 8
 * GPUs each and use one).  Rank r hashes the nonces [r 2^K / G, (r + 1) 2^K / G); buckets are owned by
 * hash range, rank g owning the buckets [g 2^B / G, (g + 1) 2^B / G) (vx_shard_owner: host arithmetic
 * only).  The exchange is fused with the first partition pass: the hashing thread claims a slot with an
 * atomic on the OWNER's partition cursor and stores the 16-byte record into the OWNER's partition array
 * through peer pointers (NVLink / NVSwitch peer access, or one device in tests) -- one all-to-all,
 * nothing staged.  After it every rank holds exactly slice r of the plot and runs
 * vx_sort_match_table2* / vx_read_tables on it as on a selected pass (no further communication).
 *   Each rank: vx_plot_create_opts(K, key, B, VX_CREATE_PASSES_LOG(log2 G)) with the SAME key, bind a
 *   workspace, then
 *     vx_shard_begin(p, r, G, stream)            zero this rank's cursors             -- BARRIER over all ranks
 *     vx_shard_scatter(p, r, G, peers, stream)   hash the share, store at the owners  -- BARRIER over all ranks
 *     vx_shard_finish(p, stream)                 scan this rank's partitions; Table 1 slice built
 *   dev_peer_workspaces[g] (HOST array of G DEVICE pointers valid on this device: the bound workspace
 *   of rank g's plot, e.g. mapped with cudaIpcOpenMemHandle; entry r is this plot's own).  The barriers
 *   (stream-complete on every rank, e.g. torch.distributed.barrier after a stream synchronize) are the
 *   caller's.  16-byte record layout only (K <= 32): VX_ERR_UNSUPPORTED in the wide layout.
 *   Measured on one device only (two workspaces standing for two peers); DESIGN.md says so. */
vx_status vx_shard_owner(uint32_t K, uint32_t bucket_bits, uint32_t world, uint32_t rank, uint64_t *nonce_begin,
                         uint64_t *nonce_end, uint64_t *bucket_begin, uint64_t *bucket_end);
vx_status vx_shard_begin(vx_plot *p, uint32_t rank, uint32_t world, void *cuda_stream);
vx_status vx_shard_scatter(vx_plot *p, uint32_t rank, uint32_t world, void *const *dev_peer_workspaces,
                           void *cuda_stream);
vx_status vx_shard_finish(vx_plot *p, void *cuda_stream);
/* Peer mapping when the ranks are separate processes (one per GPU under torch.distributed.run):
 *   vx_ipc_export  the bound workspace as a CUDA IPC handle (64 bytes, HOST) of the cudaMalloc allocation
 *                  it lies in plus its byte offset there (PyTorch's allocator sub-allocates);
 *   vx_ipc_open    in ANOTHER process: map that allocation on the current device (peer access is enabled
 *                  lazily) -> *dev_workspace for the peer table of vx_shard_scatter, *dev_mapped_base for
 *   vx_ipc_close.  The handles travel by whatever the caller has (torch.distributed.all_gather_object). */
vx_status vx_ipc_export(vx_plot *p, uint8_t handle[64], uint64_t *offset);
vx_status vx_ipc_open(const uint8_t handle[64], uint64_t offset, void **dev_mapped_base, void **dev_workspace);
vx_status vx_ipc_close(void *dev_mapped_base);

/* Copy the buckets [bucket_begin, bucket_end) of table 1 or 2 to HOST memory in the external
 * format.  Synchronises the plot's stream.  offsets_out (may be NULL) receives
 * bucket_end - bucket_begin + 1 entries relative to the first record of bucket_begin.
 * records_out == NULL only queries *records_bytes.  records_capacity is in bytes.
 * Table 1 may be read after vx_build_table1 alone (in-bucket order then unspecified, reading A9);
 * Table 2 only after vx_sort_match_table2. */
vx_status vx_read_tables(vx_plot *p, int table, uint64_t bucket_begin, uint64_t bucket_end,
                         uint64_t *offsets_out, void *records_out, size_t records_capacity,
                         size_t *records_bytes);

/* Device-side view for callers that keep the tables on the GPU (all pointers are DEVICE pointers
 * into the bound workspace; valid after vx_sort_match_table2 has completed; any may be NULL).
 *   Table 2: dev_t2_records = external 2*NONCE_SIZE-byte records, contiguous; dev_t2_offsets =
 *     uint64[2^B + 1] CSR offsets in records.
 *   Table 1 stays where stage 1 put it and is sorted IN PLACE (reading A14): dev_t1_records is the
 *     partition array of 16-byte records {uint32 H low, H high, nonce low, nonce high}, 2^pb
 *     partitions of `partition_capacity` slots each (vx_plot_info); partition q holds the buckets
 *     [q << (B - pb), (q + 1) << (B - pb)) back to back, each sorted by (H, n).  dev_t1_offsets =
 *     uint64[2^B + 1] CSR offsets in records (the numbering vx_read_tables uses) and
 *     dev_partition_base = uint64[2^pb + 1], the CSR index of each partition's first record:
 *     bucket b (partition q = b >> (B - pb)) starts at slot
 *     q * partition_capacity + dev_t1_offsets[b] - dev_partition_base[q].
 *   vx_read_tables converts to the external 12-byte Table-1 format on the way out.
 *   Wide layout (K >= 33: a 16-byte record per nonce does not fit beside Table 2 in 180 GB): same
 *     slot numbering, but dev_t1_records = uint64 a[2^pb * partition_capacity] with
 *     a = (H << pb) | (n >> t) -- the pb-bit hash prefix is the partition index, the bits it frees
 *     hold the high nonce bits -- followed (256-byte aligned) by uint16 b[] = n & (2^t - 1), t = vx_plot_layout's tile_log; sorting
 *     by (a, b) is sorting by (H, n).  dev_t2_records = uint2 {n1 & 0xffffffff, n2 & 0xffffffff},
 *     followed by uint8 hi[] = (n1 >> 32) | (n2 >> 32) << 4.  vx_read_tables converts both. */
vx_status vx_device_tables(vx_plot *p, const void **dev_t1_records, const uint64_t **dev_t1_offsets,
                           const void **dev_t2_records, const uint64_t **dev_t2_offsets,
                           const uint64_t **dev_partition_base);

/* Test hooks.  VX_OPT_FORCE_EXACT_RANK (value != 0): the fused kernel always takes the exact
 * (H, n) re-ranking path it otherwise takes only for a tile holding two equal 64-bit hashes
 * (reading A10) -- results are identical by construction; tests use it to cover that path. */
#define VX_OPT_FORCE_EXACT_RANK 1
/* VX_OPT_PARTITION_CAPACITY_LIMIT (1 .. partition_capacity) / VX_OPT_TABLE2_CAPACITY_LIMIT
 * (0 .. t2_capacity): lower the capacity the kernels CHECK against, without changing the layout,
 * so that the overflow path can be exercised: the run then ends in VX_ERR_OVERFLOW at the next
 * synchronising call instead of dropping records silently (reading A8). */
#define VX_OPT_PARTITION_CAPACITY_LIMIT 2
#define VX_OPT_TABLE2_CAPACITY_LIMIT 3
/* VX_OPT_SUBKEY_BITS (0 .. 32, default 32; 28 and above mean all 28 the kernel keeps): how many hash
 * bits below the bin index the fused kernel's fast in-bin ranking compares.  Fewer bits make records of one bin tie, come out in the wrong order
 * and so send the tile through its "redo with exact (H, n) ranks" path (taken by about 8 tiles of
 * a K = 31 plot otherwise) -- results are identical by construction; tests use it to run that path. */
#define VX_OPT_SUBKEY_BITS 4
/* VX_OPT_STAGE2_KERNEL (0, default: the fused kernel whose phases are separated by CTA-wide barriers; 1: the
 * warp-local variant, in which from the scatter on every warp finishes its own hash range of the tile alone,
 * wherever it applies -- narrow layout, a warp's range a whole number of buckets: K = 27 .. 32 at B = 24 -- and
 * the default kernel elsewhere).  Results are identical; the variant measured slower and is kept
 * as a measured alternative.  Tests and measurements use the option to run both. */
#define VX_OPT_STAGE2_KERNEL 5
vx_status vx_plot_set_option(vx_plot *p, int option, uint64_t value);

/* Synchronises; any output pointer may be NULL.  max_bucket = largest Table-1 bucket. */
vx_status vx_get_stats(vx_plot *p, uint64_t *t1_records, uint64_t *t2_records, uint32_t *max_bucket);

/* Synchronises.  tile_retries = tiles of the last stage 2 whose fast in-bin ranking met a tie (two
 * records of a bin with equal compared sub-keys, among them equal 64-bit hashes, reading A10) and
 * which were therefore re-ranked by exact (H, n) compares; about 2^-16 per tile at the default
 * sub-key bits.  For tests of that path (VX_OPT_SUBKEY_BITS). */
vx_status vx_get_counters(vx_plot *p, uint64_t *tile_retries);

/* Wait for the plot's enqueued work and report device-raised errors. */
vx_status vx_synchronize(vx_plot *p);

/* Hash kernel alone (7 build-plan step 3): H(n) for
 * n in [nonce_begin, nonce_begin + count) written as uint64 to dev_hashes[count].  Enqueues only. */
vx_status vx_hash_range(vx_plot *p, uint64_t nonce_begin, uint64_t count, uint64_t *dev_hashes,
                        void *cuda_stream);

/* Measurement aid for the ALU roofline: hashes `count` nonces starting at 0 and folds them into
 * one xor word per thread block (dev_sink[grid] uint64) -- the BLAKE3 stage with no table traffic. */
vx_status vx_hash_sink(vx_plot *p, uint64_t count, uint64_t *dev_sink, size_t sink_words,
                       void *cuda_stream);

/* The same fold for callers that cannot allocate (code under CUDA graph capture, tight serving loops,
 * harnesses that forbid cudaMalloc): hashes the nonces [nonce_begin, nonce_begin + count) and writes the
 * xor of their hashes to dev_out[0] (DEVICE, one uint64).  Its scratch -- one partial word per thread
 * block -- is a file-scope device array of libvx.so (256 KB, held by every GPU that loads the library
 * until the process exits), so the call allocates nothing: no cudaMalloc, cudaFree or allocating library
 * routine, and the plot need not be bound.  Limit: count <= 2^25 nonces per call, VX_ERR_RANGE beyond
 * (text in vx_last_error).  Every call on a device shares that array: calls that overlap on the GPU
 * (different streams or host threads) race -- serialise them on one stream.  Enqueues only. */
vx_status vx_hash_fold_noalloc(vx_plot *p, uint64_t nonce_begin, uint64_t count, uint64_t *dev_out,
                               void *cuda_stream);

/* Measurement aid for the same roofline (the integer pipes' issue rate is not in
 * MEASURED_PEAKS.json and is to be measured with dependent-free instruction chains): launches
 * vx_sm_count x ctas_per_sm CTAs of 256 threads, each thread running 8 independent chains of
 * 8 * iters instructions of one kind; *lane_ops = thread-instructions of that kind executed.
 * dev_out: DEVICE scratch of >= 1024 uint32.  Enqueues only; the caller times it with CUDA events. */
#define VX_PROBE_LOP3 0 /* a = a ^ b ^ c            (ALU pipe)                 */
#define VX_PROBE_SHF 1  /* rotate                   (ALU pipe)                 */
#define VX_PROBE_ADD 2  /* 32-bit add               (ptxas: IADD3 or IMAD.IADD) */
#define VX_PROBE_IMAD 3 /* a = a * b + c            (FMA pipe)                 */
#define VX_PROBE_PRMT 4 /* byte permute             (ALU pipe)                 */
#define VX_PROBE_ARX 5  /* xor, rotate alternating  (BLAKE3's mix)             */
vx_status vx_probe_alu(int kind, uint32_t iters, uint32_t ctas_per_sm, uint32_t *dev_out, size_t out_words,
                       void *cuda_stream, uint64_t *lane_ops);

/* Plot geometry, for tests and the bench report.  Any pointer may be NULL. */
vx_status vx_plot_info(const vx_plot *p, uint32_t *K, uint32_t *bucket_bits, uint32_t *nonce_size,
                       uint32_t *partition_bits, uint32_t *partition_capacity, uint64_t *t2_capacity);

/* Internal layout, for callers of vx_device_tables: wide = 1 for the 10-byte Table-1 layout;
 * tile_log = log2 of the mean partition size (12 for K <= 31, 13 from K = 32). */
vx_status vx_plot_layout(const vx_plot *p, uint32_t *wide, uint32_t *tile_log);

/* Kernels one vx_build_table1 / vx_sort_match_table2 call launches (for the bench report's
 * gpu_launches): 3 (clear, hash+scatter, partition scan) + 2 (clear, fused sort+match) in the narrow
 * layout; the wide layout builds Table 1 in 4 rounds of hash+scatter and compaction
 * (DESIGN.md "stage 1 in rounds"): 2 clears + 2 * 4 + 1 launches. */
vx_status vx_plot_launches(const vx_plot *p, uint32_t *build_table1, uint32_t *sort_match_table2);

const char *vx_last_error(const vx_plot *p); /* never NULL; includes cudaGetErrorString text */
const char *vx_status_string(vx_status s);
void vx_free(vx_plot *p);                     /* frees the handle, never the workspace */

#ifdef __cplusplus
}
#endif
#endif /* VX_H_ */
