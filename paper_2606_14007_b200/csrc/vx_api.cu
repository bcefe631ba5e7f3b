// vx_api.cu -- the C ABI of libvx (include/vx.h): host-side state machine, workspace plan,
// launches and read-back.  No device memory is allocated here: the workspace is the caller's.
#include <dlfcn.h>
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>
#include <unistd.h>

#include <atomic>
#include <mutex>
#include <new>

#include "../../include/vx.h"
#include "vx_internal.h"

enum VxState { VX_CREATED = 0, VX_BOUND = 1, VX_BUILT = 2, VX_MATCHED = 3, VX_REKEYED = 4 };

struct vx_plot {
    VxGeom g;
    VxHashConst hc;
    VxHashConst hc2;        // the same key with block_len = 2 NONCE_SIZE: the pair hash of the re-keying (A19)
    uint8_t key[32];
    uint8_t *ws;
    size_t ws_bytes;
    VxState state;
    bool t1_materialised;   // the 2^B-bucket view of Table 1 exists in the workspace
    bool force_exact;       // VX_OPT_FORCE_EXACT_RANK
    cudaStream_t stream;    // stream of the last enqueue
    int num_sms;
    char err[512];
};

static size_t align256(size_t x) { return (x + 255) & ~(size_t)255; }

// ------------------------------------------------------------------------------ geometry
void vx_geom_select_pass(VxGeom *g, uint32_t pass)
{
    g->pass = pass;
    g->p_first = (uint64_t)pass * g->P;
    g->b_first = (uint64_t)pass * g->NBp;
}

bool vx_geom_init(VxGeom *g, uint32_t K, uint32_t B, bool force_wide, bool force_big_tiles, uint32_t passes_log)
{
    memset(g, 0, sizeof *g);
    if (K < 1 || K > VX_MAX_K || B < 1 || B > 24) return false;
    if (passes_log > VX_MAX_PASSES_LOG) return false;
    if (K > B + VX_MAX_MEAN_BUCKET_LOG + passes_log) return false;
    g->K = K; g->B = B;
    g->nonce_size = K <= 32 ? 4 : 5;                       // reading A1
    g->wide = (g->nonce_size > 4 || force_wide) ? 1u : 0u;
    g->tile_log = (K >= VX_BIG_TILES_FROM_K || force_big_tiles) ? VX_TILE_LOG_BIG : VX_TILE_LOG;
    g->pb = K > g->tile_log ? K - g->tile_log : 0;
    if (g->pb > B) return false;                           // cannot happen while K - B <= 9
    g->fb = B - g->pb;
    if (passes_log > g->pb || passes_log > B) return false;  // a pass is a whole number of partitions (and buckets)
    g->passes_log = passes_log;
    g->N = 1ull << K; g->P = 1ull << (g->pb - passes_log); g->NB = 1ull << B;
    g->NBp = g->NB >> passes_log;
    vx_geom_select_pass(g, 0);
    const uint64_t mean = g->N >> g->pb;
    uint64_t cap;
    // Poisson tail, 8 sigma.  Also with a single partition (pb = 0), which holds exactly 2^K records in
    // stage 1: the re-keying appends |Table 2| records to the same partitions, and |Table 2| can exceed 2^K
    // by a few sigma when K is tiny
    cap = mean + (uint64_t)ceil(8.0 * sqrt((double)mean));
    cap = (cap + 31) & ~(uint64_t)31;
    if (cap > (g->tile_log == VX_TILE_LOG_BIG ? VX_S2B_THREADS * VX_S2B_ITEMS : VX_S2_THREADS * VX_S2_ITEMS)) return false;
    g->cap = (uint32_t)cap;
    g->cap_check = g->cap;
    // |T2| ~ 2^K (1 - 2^(B-K-1)) for K >= B, 2^(2K-1-B) below; sd ~ sqrt: 2^K + slack is ample
    g->t2_cap = (g->N >> passes_log) + (1u << 16);        // per pass
    g->t2_check = g->t2_cap;
    g->subkey_bits = 32;
    g->s2_kernel = 0;
    g->rec1_bytes = g->nonce_size + 8;
    g->rec2_bytes = 2 * g->nonce_size;
    size_t o = 0;
    g->off_ctrl = o;      o = align256(o + sizeof(VxCtrl));
    g->off_cursor = o;    o = align256(o + g->P * 4);
    g->off_part_base = o; o = align256(o + (g->P + 1) * 8);
    g->off_status = o;    o = align256(o + g->P * 8);
    if (!g->wide) {
        g->off_part = o;  o = align256(o + g->P * (size_t)g->cap * 16);
    } else {
        g->off_part = o;   o = align256(o + g->P * (size_t)g->cap * 8);
        g->off_part_b = o; o = align256(o + g->P * (size_t)g->cap * 2);
    }
    g->off_t1_off = o;    o = align256(o + (g->NBp + 1) * 8);
    g->off_t2_off = o;    o = align256(o + (g->NBp + 1) * 8);
    size_t t2_bytes = g->t2_cap * (size_t)8;
    if (g->wide) {
        // stage 1 in rounds: 4 slices (K >= 2), scratch partitions one hash bit coarser than the
        // final ones.  K = 33: slices of 2^31 nonces into 2^19 scratch partitions of ~4096 records,
        // the geometry stage 1 runs ALU-bound in at K = 31.
        g->round_log = K >= 2 ? K - 2 : K;
        g->rounds = 1u << (K - g->round_log);
        g->pb_tmp = g->pb > passes_log ? g->pb - 1 : g->pb;     // (global bit count, like pb)
        const uint64_t mean_tmp = (1ull << g->round_log) >> g->pb_tmp;
        uint64_t cap_tmp = (g->pb_tmp == 0 && passes_log == 0) ? mean_tmp : mean_tmp + (uint64_t)ceil(8.0 * sqrt((double)mean_tmp));
        cap_tmp = (cap_tmp + 31) & ~(uint64_t)31;
        g->cap_tmp = (uint32_t)cap_tmp;
        const size_t tmp_bytes = ((size_t)1 << (g->pb_tmp - passes_log)) * cap_tmp * 16;
        if (tmp_bytes > t2_bytes) t2_bytes = tmp_bytes;      // tiny K only
        g->off_cursor_tmp = o; o = align256(o + ((size_t)4 << (g->pb_tmp - passes_log)));
    }
    o = (o + ((size_t)2 << 20) - 1) & ~(((size_t)2 << 20) - 1);   // Table 2 on a 2 MB boundary: D2H copies of it run faster aligned
    g->off_t2_rec = o;    o = align256(o + t2_bytes);
    g->off_tmp = g->off_t2_rec;                              // scratch of stage 1, dead before stage 2
    if (g->wide) { g->off_t2_hi = o; o = align256(o + g->t2_cap); }
    g->stage_bytes = (g->N >> passes_log) * (size_t)g->rec1_bytes;
    if (g->stage_bytes > VX_STAGE_MAX_BYTES) g->stage_bytes = VX_STAGE_MAX_BYTES;
    g->off_stage = o;     o = align256(o + g->stage_bytes);
    g->total = o;
    return true;
}

// ------------------------------------------------------------------------------ host fold
// BLAKE3 G function on the host, used once per plot for the three nonce-independent columns of
// round 1 (message words 2..7 are zero for a nonce of at most 5 bytes).  BLAKE3 spec 2.2.
static uint32_t h_rotr(uint32_t x, int r) { return (x >> r) | (x << (32 - r)); }
static void h_g0(uint32_t &a, uint32_t &b, uint32_t &c, uint32_t &d)
{
    a = a + b;  d = h_rotr(d ^ a, 16);  c = c + d;  b = h_rotr(b ^ c, 12);
    a = a + b;  d = h_rotr(d ^ a, 8);   c = c + d;  b = h_rotr(b ^ c, 7);
}

void vx_hash_const_init(VxHashConst *hc, const uint8_t key[32], uint32_t nonce_size)
{
    const uint32_t iv[4] = {VX_IV0, VX_IV1, VX_IV2, VX_IV3};
    for (int i = 0; i < 8; i++)
        hc->k[i] = (uint32_t)key[4 * i] | ((uint32_t)key[4 * i + 1] << 8) |
                   ((uint32_t)key[4 * i + 2] << 16) | ((uint32_t)key[4 * i + 3] << 24);
    hc->s04 = hc->k[0] + hc->k[4];
    hc->block_len = nonce_size;
    // v12 = v13 = 0 (counter), v14 = block_len, v15 = flags
    const uint32_t tail[4] = {0u, 0u, nonce_size, VX_FLAGS};
    for (int c = 1; c < 4; c++) {
        uint32_t a = hc->k[c], b = hc->k[4 + c], cc = iv[c], d = tail[c];
        h_g0(a, b, cc, d);
        hc->col[4 * (c - 1) + 0] = a;
        hc->col[4 * (c - 1) + 1] = b;
        hc->col[4 * (c - 1) + 2] = cc;
        hc->col[4 * (c - 1) + 3] = d;
    }
}

// ------------------------------------------------------------------------------ helpers
int vx_sm_count(void)
{
    static std::atomic<int> cache[64];
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return 148;
    if (dev >= 0 && dev < 64 && (sms = cache[dev].load(std::memory_order_relaxed)) > 0) return sms;
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms <= 0) return 148;
    if (dev >= 0 && dev < 64) cache[dev].store(sms, std::memory_order_relaxed);
    return sms;
}

static vx_status fail(vx_plot *p, vx_status s, const char *what)
{
    if (p) snprintf(p->err, sizeof p->err, "%s: %s", vx_status_string(s), what);
    return s;
}

static vx_status fail_cuda(vx_plot *p, cudaError_t e, const char *what)
{
    if (p) snprintf(p->err, sizeof p->err, "VX_ERR_CUDA: %s: %s", what, cudaGetErrorString(e));
    return VX_ERR_CUDA;
}

static vx_status sync_and_check(vx_plot *p)
{
    cudaError_t e = cudaStreamSynchronize(p->stream);
    if (e != cudaSuccess) return fail_cuda(p, e, "cudaStreamSynchronize");
    if (p->state >= VX_BUILT) {
        VxCtrl c;
        e = cudaMemcpy(&c, p->ws + p->g.off_ctrl, sizeof c, cudaMemcpyDeviceToHost);
        if (e != cudaSuccess) return fail_cuda(p, e, "cudaMemcpy(ctrl)");
        if (c.flags & VX_FLAG_BOUNDS)
            return fail(p, VX_ERR_CUDA, "internal bounds check failed (VX_DEBUG_BOUNDS build)");
        if (c.flags & VX_FLAG_PART_OVERFLOW)
            return fail(p, VX_ERR_OVERFLOW, "a stage-1 partition exceeded its slack capacity");
        if (c.flags & VX_FLAG_T2_OVERFLOW)
            return fail(p, VX_ERR_OVERFLOW, "Table 2 exceeded its capacity");
    }
    return VX_OK;
}

const VxHashConst &vx_plot_hash_const(const vx_plot *p) { return p->hc; }
int vx_plot_fail(vx_plot *p, int status, const char *what) { return fail(p, (vx_status)status, what); }
int vx_plot_fail_cuda(vx_plot *p, cudaError_t e, const char *what) { return fail_cuda(p, e, what); }

// ------------------------------------------------------------------------------ the ABI
extern "C" {

const char *vx_status_string(vx_status s)
{
    switch (s) {
    case VX_OK: return "VX_OK";
    case VX_ERR_ARG: return "VX_ERR_ARG";
    case VX_ERR_STATE: return "VX_ERR_STATE";
    case VX_ERR_WORKSPACE: return "VX_ERR_WORKSPACE";
    case VX_ERR_CUDA: return "VX_ERR_CUDA";
    case VX_ERR_OVERFLOW: return "VX_ERR_OVERFLOW";
    case VX_ERR_RANGE: return "VX_ERR_RANGE";
    case VX_ERR_UNSUPPORTED: return "VX_ERR_UNSUPPORTED";
    case VX_ERR_IO: return "VX_ERR_IO";
    case VX_ERR_NOMEM: return "VX_ERR_NOMEM";
    }
    return "VX_ERR_?";
}

// flags -> geometry.  Passes: the explicit VX_CREATE_PASSES_LOG field, else the fewest passes that keep
// at most 2^33 records resident (K <= 33: one pass).
static bool geom_from_flags(VxGeom *g, uint32_t K, uint32_t bucket_bits, uint32_t flags)
{
    if (flags & ~(uint32_t)(VX_CREATE_WIDE_LAYOUT | VX_CREATE_BIG_TILES | VX_CREATE_PASSES_LOG_MASK)) return false;
    uint32_t pl = (flags & VX_CREATE_PASSES_LOG_MASK) >> VX_CREATE_PASSES_LOG_SHIFT;
    if (pl == 0 && K > bucket_bits + VX_MAX_MEAN_BUCKET_LOG && bucket_bits == 24) pl = K - bucket_bits - VX_MAX_MEAN_BUCKET_LOG;
    return vx_geom_init(g, K, bucket_bits, (flags & VX_CREATE_WIDE_LAYOUT) != 0, (flags & VX_CREATE_BIG_TILES) != 0, pl);
}

size_t vx_workspace_bytes_opts(uint32_t K, uint32_t bucket_bits, uint32_t flags)
{
    VxGeom g;
    if (!geom_from_flags(&g, K, bucket_bits, flags)) return 0;
    return g.total;
}

size_t vx_workspace_bytes_ex(uint32_t K, uint32_t bucket_bits) { return vx_workspace_bytes_opts(K, bucket_bits, 0); }

size_t vx_workspace_bytes(uint32_t K) { return vx_workspace_bytes_opts(K, 24, 0); }

vx_status vx_plot_create_opts(uint32_t K, const uint8_t key[32], uint32_t bucket_bits, uint32_t flags,
                              vx_plot **out)
{
    if (!out) return VX_ERR_ARG;
    *out = NULL;
    if (!key) return VX_ERR_ARG;
    VxGeom g;
    if (!geom_from_flags(&g, K, bucket_bits, flags)) return VX_ERR_ARG;
    vx_plot *p = new (std::nothrow) vx_plot;
    if (!p) return VX_ERR_NOMEM;
    memset(p, 0, sizeof *p);
    p->g = g;
    memcpy(p->key, key, 32);
    vx_hash_const_init(&p->hc, key, g.nonce_size);
    vx_hash_const_init(&p->hc2, key, 2 * g.nonce_size);
    p->state = VX_CREATED;
    snprintf(p->err, sizeof p->err, "VX_OK");
    *out = p;
    return VX_OK;
}

vx_status vx_plot_create_ex(uint32_t K, const uint8_t key[32], uint32_t bucket_bits, vx_plot **out)
{
    return vx_plot_create_opts(K, key, bucket_bits, 0, out);
}

vx_status vx_plot_create(uint32_t K, const uint8_t key[32], vx_plot **out)
{
    return vx_plot_create_ex(K, key, 24, out);
}

vx_status vx_plot_bind(vx_plot *p, void *dev_workspace, size_t bytes)
{
    if (!p || !dev_workspace) return fail(p, VX_ERR_ARG, "NULL plot or workspace");
    if (((uintptr_t)dev_workspace & 255) != 0) return fail(p, VX_ERR_WORKSPACE, "workspace not 256-byte aligned");
    if (bytes < p->g.total) return fail(p, VX_ERR_WORKSPACE, "workspace smaller than vx_workspace_bytes");
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return fail_cuda(p, e, "cudaGetDevice (no CUDA device: there is no CPU fallback)");
    // attributes, not cudaGetDeviceProperties: that call takes 3-12 ms, and a plot is bound per key
    int major = 0, sms = 0;
    e = cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (e != cudaSuccess) return fail_cuda(p, e, "cudaDeviceGetAttribute");
    if (major < 10) return fail(p, VX_ERR_CUDA, "libvx is built for sm_100a only");
    p->num_sms = sms;
    {
        static std::mutex mu;                              // plots are bound from several host threads
        static uint64_t configured = 0;                    // one bit per device ordinal < 64
        std::lock_guard<std::mutex> lock(mu);
        if (dev >= 64 || !(configured & (1ull << dev))) {
            e = vx_stage2_configure();
            if (e != cudaSuccess) return fail_cuda(p, e, "cudaFuncSetAttribute(stage 2 shared memory)");
            if (dev < 64) configured |= 1ull << dev;
        }
    }
    p->ws = (uint8_t *)dev_workspace;
    p->ws_bytes = bytes;
    p->state = VX_BOUND;
    p->t1_materialised = false;
    p->stream = 0;
    return VX_OK;
}

vx_status vx_build_table1(vx_plot *p, void *cuda_stream)
{
    if (!p) return VX_ERR_ARG;
    if (p->state < VX_BOUND) return fail(p, VX_ERR_STATE, "vx_build_table1 before vx_plot_bind");
    p->stream = (cudaStream_t)cuda_stream;
    cudaError_t e = vx_launch_stage1(p->g, p->hc, p->ws, p->stream);
    if (e != cudaSuccess) return fail_cuda(p, e, "stage 1 launch");
    p->state = VX_BUILT;
    p->t1_materialised = false;
    return VX_OK;
}

vx_status vx_sort_match_table2(vx_plot *p, void *cuda_stream)
{
    if (!p) return VX_ERR_ARG;
    if (p->state < VX_BUILT) return fail(p, VX_ERR_STATE, "vx_sort_match_table2 before vx_build_table1");
    p->stream = (cudaStream_t)cuda_stream;
    cudaError_t e = vx_launch_stage2(p->g, p->ws, true, p->force_exact, p->num_sms, p->stream);
    if (e != cudaSuccess) return fail_cuda(p, e, "stage 2 launch");
    p->state = VX_MATCHED;
    p->t1_materialised = true;
    return VX_OK;
}

vx_status vx_synchronize(vx_plot *p)
{
    if (!p) return VX_ERR_ARG;
    if (p->state < VX_BOUND) return fail(p, VX_ERR_STATE, "vx_synchronize before vx_plot_bind");
    return sync_and_check(p);
}

vx_status vx_read_tables(vx_plot *p, int table, uint64_t bucket_begin, uint64_t bucket_end,
                         uint64_t *offsets_out, void *records_out, size_t records_capacity,
                         size_t *records_bytes)
{
    if (!p) return VX_ERR_ARG;
    if (table != 1 && table != 2 && table != VX_TABLE2_REKEYED) return fail(p, VX_ERR_ARG, "table must be 1, 2 or VX_TABLE2_REKEYED");
    if (p->state < VX_BUILT) return fail(p, VX_ERR_STATE, "vx_read_tables before vx_build_table1");
    if (table == 2 && p->state < VX_MATCHED)
        return fail(p, VX_ERR_STATE, "Table 2 read before vx_sort_match_table2");
    if (table == VX_TABLE2_REKEYED && p->state < VX_REKEYED)
        return fail(p, VX_ERR_STATE, "re-keyed Table 2 read before vx_rekey_table2");
    if (table == 1 && p->state >= VX_REKEYED)
        return fail(p, VX_ERR_STATE, "Table 1 was overwritten by vx_rekey_table2 (its partition array holds the pair hashes now)");
    if (bucket_begin > bucket_end || bucket_end > p->g.NB)
        return fail(p, VX_ERR_RANGE, "bucket range outside [0, 2^B]");
    if (bucket_begin < p->g.b_first || bucket_end > p->g.b_first + p->g.NBp)
        return fail(p, VX_ERR_RANGE, "bucket range outside the selected pass (vx_plot_select_pass)");
    bucket_begin -= p->g.b_first;                          // offsets in the workspace are relative to the pass
    bucket_end -= p->g.b_first;
    if (!p->t1_materialised) {
        // Table 1 read after stage 1 alone: split the partitions into buckets now (no matching)
        cudaError_t e = vx_launch_stage2(p->g, p->ws, false, p->force_exact, p->num_sms, p->stream);
        if (e != cudaSuccess) return fail_cuda(p, e, "stage 2 (bucket view) launch");
        p->t1_materialised = true;
    }
    vx_status s = sync_and_check(p);
    if (s != VX_OK) return s;
    // (the re-keyed table's CSR offsets were written where Table 1's were)
    const uint8_t *off_dev = p->ws + (table == 2 ? p->g.off_t2_off : p->g.off_t1_off);
    const size_t rb = table == 1 ? p->g.rec1_bytes : p->g.rec2_bytes;
    const uint64_t nb = bucket_end - bucket_begin;
    uint64_t first = 0, last = 0;
    cudaError_t e = cudaMemcpy(&first, off_dev + bucket_begin * 8, 8, cudaMemcpyDeviceToHost);
    if (e == cudaSuccess) e = cudaMemcpy(&last, off_dev + bucket_end * 8, 8, cudaMemcpyDeviceToHost);
    if (e != cudaSuccess) return fail_cuda(p, e, "cudaMemcpy(offsets ends)");
    const size_t need = (size_t)(last - first) * rb;
    if (records_bytes) *records_bytes = need;
    if (offsets_out) {
        e = cudaMemcpy(offsets_out, off_dev + bucket_begin * 8, (nb + 1) * 8, cudaMemcpyDeviceToHost);
        if (e != cudaSuccess) return fail_cuda(p, e, "cudaMemcpy(offsets)");
        for (uint64_t i = 0; i <= nb; i++) offsets_out[i] -= first;
    }
    if (!records_out) return VX_OK;
    if (records_capacity < need) return fail(p, VX_ERR_RANGE, "records_capacity too small");
    if (need == 0) return VX_OK;
    if (table == 2 && p->g.nonce_size > 4) {
        // wide records (n1 lo, n2 lo) + high-bits byte -> external 10-byte records through staging
        const uint64_t per2 = p->g.stage_bytes / rb;
        for (uint64_t done = 0; done < last - first; done += per2) {
            const uint64_t n = (last - first - done) < per2 ? (last - first - done) : per2;
            e = vx_launch_export_t2(p->g, p->ws, first + done, n, p->stream);
            if (e != cudaSuccess) return fail_cuda(p, e, "export launch");
            e = cudaMemcpyAsync((uint8_t *)records_out + done * rb, p->ws + p->g.off_stage, n * rb,
                                cudaMemcpyDeviceToHost, p->stream);
            if (e == cudaSuccess) e = cudaStreamSynchronize(p->stream);
            if (e != cudaSuccess) return fail_cuda(p, e, "cudaMemcpy(exported records)");
        }
        return VX_OK;
    }
    if (table == VX_TABLE2_REKEYED) {
        // gather the pairs in H2 order through the sorted pair indices, a staging chunk at a time
        const uint64_t per3 = p->g.stage_bytes / rb;
        for (uint64_t done = 0; done < last - first; done += per3) {
            const uint64_t n = (last - first - done) < per3 ? (last - first - done) : per3;
            e = vx_launch_export_rekey(p->g, p->ws, first + done, n, p->stream);
            if (e != cudaSuccess) return fail_cuda(p, e, "export launch");
            e = cudaMemcpyAsync((uint8_t *)records_out + done * rb, p->ws + p->g.off_stage, n * rb,
                                cudaMemcpyDeviceToHost, p->stream);
            if (e == cudaSuccess) e = cudaStreamSynchronize(p->stream);
            if (e != cudaSuccess) return fail_cuda(p, e, "cudaMemcpy(exported records)");
        }
        return VX_OK;
    }
    if (table == 2) {
        // Table 2 is resident in the external format (4-byte nonces): one contiguous copy
        e = cudaMemcpy(records_out, p->ws + p->g.off_t2_rec + (size_t)first * rb, need, cudaMemcpyDeviceToHost);
        if (e != cudaSuccess) return fail_cuda(p, e, "cudaMemcpy(records)");
        return VX_OK;
    }
    // Table 1 is resident as sorted buckets inside the partition array (16-byte internal records):
    // gather + convert to the external format through the staging area, a chunk at a time
    const uint64_t per = p->g.stage_bytes / rb;
    for (uint64_t done = 0; done < last - first; done += per) {
        const uint64_t n = (last - first - done) < per ? (last - first - done) : per;
        e = vx_launch_export_t1(p->g, p->ws, first + done, n, p->stream);
        if (e != cudaSuccess) return fail_cuda(p, e, "export launch");
        e = cudaMemcpyAsync((uint8_t *)records_out + done * rb, p->ws + p->g.off_stage, n * rb,
                            cudaMemcpyDeviceToHost, p->stream);
        if (e == cudaSuccess) e = cudaStreamSynchronize(p->stream);
        if (e != cudaSuccess) return fail_cuda(p, e, "cudaMemcpy(exported records)");
    }
    return VX_OK;
}

// ------------------------------------------------------------------------------ egress (8(f1))
static vx_status egress_common(vx_plot *p, void *compute_stream, void *copy_stream, uint32_t slices,
                               uint8_t *host_records, size_t records_capacity, uint64_t *host_offsets,
                               VxRing *ring, uint64_t *t2_records)
{
    if (p->state < VX_BUILT) return fail(p, VX_ERR_STATE, "Table-2 egress before vx_build_table1");
    if (compute_stream == copy_stream) return fail(p, VX_ERR_ARG, "compute and copy streams must differ");
    p->stream = (cudaStream_t)compute_stream;
    int soft = 0;
    char msg[256] = "";
    VxCtrl ctrl;
    memset(&ctrl, 0, sizeof ctrl);
    cudaError_t e = vx_egress_run(p->g, p->ws, p->force_exact, p->num_sms, p->stream, (cudaStream_t)copy_stream,
                                  slices, host_records, records_capacity, host_offsets, ring, t2_records, &ctrl,
                                  &soft, msg, sizeof msg);
    if (e != cudaSuccess) return fail_cuda(p, e, "Table-2 egress");
    p->state = VX_MATCHED;
    p->t1_materialised = true;
    if (soft == 1) return fail(p, VX_ERR_RANGE, msg);
    if (soft == 2) return fail(p, VX_ERR_OVERFLOW, msg);
    if (soft == 3) return fail(p, VX_ERR_IO, msg);
    if (soft == 4) return fail(p, VX_ERR_UNSUPPORTED, msg);
    // both streams have drained inside vx_egress_run; the flags came back through the mailbox
    if (ctrl.flags & VX_FLAG_BOUNDS)
        return fail(p, VX_ERR_CUDA, "internal bounds check failed (VX_DEBUG_BOUNDS build)");
    if (ctrl.flags & VX_FLAG_PART_OVERFLOW)
        return fail(p, VX_ERR_OVERFLOW, "a stage-1 partition exceeded its slack capacity");
    if (ctrl.flags & VX_FLAG_T2_OVERFLOW)
        return fail(p, VX_ERR_OVERFLOW, "Table 2 exceeded its capacity");
    return VX_OK;
}

vx_status vx_sort_match_table2_to_host(vx_plot *p, void *compute_stream, void *copy_stream, uint32_t slices,
                                       void *host_records, size_t records_capacity, uint64_t *host_offsets,
                                       size_t *records_bytes)
{
    if (!p) return VX_ERR_ARG;
    if (!host_records) return fail(p, VX_ERR_ARG, "NULL host_records");
    uint64_t n = 0;
    vx_status s = egress_common(p, compute_stream, copy_stream, slices, (uint8_t *)host_records, records_capacity,
                                host_offsets, NULL, &n);
    if (records_bytes) *records_bytes = (size_t)n * p->g.rec2_bytes;
    return s;
}

vx_status vx_sort_match_table2_to_file(vx_plot *p, void *compute_stream, void *copy_stream, uint32_t slices,
                                       int fd, void *pinned_staging, size_t staging_bytes, uint64_t *file_bytes)
{
    if (!p) return VX_ERR_ARG;
    if (fd < 0 || !pinned_staging) return fail(p, VX_ERR_ARG, "bad file descriptor or NULL staging buffer");
    VxRing *ring = vx_ring_create(pinned_staging, staging_bytes, fd);
    if (!ring) return fail(p, VX_ERR_ARG, "staging buffer smaller than two 4 MB chunks");
    uint64_t n = 0;
    vx_status s = egress_common(p, compute_stream, copy_stream, slices, NULL, 0, NULL, ring, &n);
    uint64_t written = vx_ring_written(ring);
    vx_ring_destroy(ring);
    if (s == VX_OK) {
        // trailer: magic, K, B, NONCE_SIZE, reserved, |Table 2|  (all little-endian)
        uint8_t tr[32] = {'V', 'X', 'T', '2', 0, 0, 0, 1};
        // (a plot made in passes: this file is the selected pass's slice; the last word says which of how many)
        const uint32_t w[4] = {p->g.K, p->g.B, p->g.nonce_size, p->g.pass | (p->g.passes_log << 16)};
        memcpy(tr + 8, w, 16);
        memcpy(tr + 24, &n, 8);
        char msg[128];
        if (vx_write_all(fd, tr, sizeof tr, &written, msg, sizeof msg)) s = fail(p, VX_ERR_IO, msg);
    }
    if (file_bytes) *file_bytes = written;
    return s;
}

// ------------------------------------------------------------------------------ re-keying + plot file (8(f2))
vx_status vx_rekey_table2(vx_plot *p, void *cuda_stream)
{
    if (!p) return VX_ERR_ARG;
    if (p->state < VX_MATCHED) return fail(p, VX_ERR_STATE, "vx_rekey_table2 before vx_sort_match_table2");
    if (p->state >= VX_REKEYED) return fail(p, VX_ERR_STATE, "Table 2 is already re-keyed");
    if (p->g.passes_log)
        return fail(p, VX_ERR_UNSUPPORTED, "re-keying needs the whole of Table 2 resident: one-pass plots only (K <= 33)");
    p->stream = (cudaStream_t)cuda_stream;
    cudaError_t e = vx_launch_rekey(p->g, p->hc2, p->ws, p->stream);
    if (e == cudaSuccess) e = vx_launch_stage2(p->g, p->ws, false, p->force_exact, p->num_sms, p->stream);
    if (e != cudaSuccess) return fail_cuda(p, e, "re-keying launch");
    p->state = VX_REKEYED;
    p->t1_materialised = true;                             // the bucket view in the workspace is the re-keyed table's
    return VX_OK;
}

vx_status vx_write_plot_file(vx_plot *p, int fd, void *pinned_staging, size_t staging_bytes, uint64_t *file_bytes)
{
    if (!p) return VX_ERR_ARG;
    if (file_bytes) *file_bytes = 0;
    if (fd < 0 || !pinned_staging || staging_bytes < ((size_t)1 << 20))
        return fail(p, VX_ERR_ARG, "bad file descriptor, or staging buffer NULL / smaller than 1 MB");
    if (p->state < VX_REKEYED) return fail(p, VX_ERR_STATE, "vx_write_plot_file before vx_rekey_table2");
    vx_status s = sync_and_check(p);
    if (s != VX_OK) return s;
    VxCtrl c;
    cudaError_t e = cudaMemcpy(&c, p->ws + p->g.off_ctrl, sizeof c, cudaMemcpyDeviceToHost);
    if (e != cudaSuccess) return fail_cuda(p, e, "cudaMemcpy(ctrl)");
    const uint64_t M = c.t2_total;
    uint64_t written = 0;
    char msg[128];
    // header (reading A21): magic, K, B, NONCE_SIZE, 0, key, record count
    uint8_t hd[64] = {'V', 'X', 'P', 'L', 'O', 'T', 0, 1};
    const uint32_t w[4] = {p->g.K, p->g.B, p->g.nonce_size, 0u};
    memcpy(hd + 8, w, 16);
    memcpy(hd + 24, p->key, 32);
    memcpy(hd + 56, &M, 8);
    if (vx_write_all(fd, hd, sizeof hd, &written, msg, sizeof msg)) return fail(p, VX_ERR_IO, msg);
    uint8_t *host = (uint8_t *)pinned_staging;
    // CSR offsets, then the records in H2 order (gathered on the device a staging chunk at a time)
    const uint8_t *off_dev = p->ws + p->g.off_t1_off;
    const size_t off_bytes = (p->g.NB + 1) * 8;
    for (size_t at = 0; at < off_bytes; at += staging_bytes) {
        const size_t n = off_bytes - at < staging_bytes ? off_bytes - at : staging_bytes;
        e = cudaMemcpy(host, off_dev + at, n, cudaMemcpyDeviceToHost);
        if (e != cudaSuccess) return fail_cuda(p, e, "cudaMemcpy(offsets)");
        if (vx_write_all(fd, host, n, &written, msg, sizeof msg)) { if (file_bytes) *file_bytes = written; return fail(p, VX_ERR_IO, msg); }
    }
    const size_t rb = p->g.rec2_bytes;
    size_t chunk = (p->g.stage_bytes < staging_bytes ? p->g.stage_bytes : staging_bytes) / rb;
    for (uint64_t done = 0; done < M; done += chunk) {
        const uint64_t n = M - done < chunk ? M - done : chunk;
        e = vx_launch_export_rekey(p->g, p->ws, done, n, p->stream);
        if (e == cudaSuccess) e = cudaMemcpyAsync(host, p->ws + p->g.off_stage, n * rb, cudaMemcpyDeviceToHost, p->stream);
        if (e == cudaSuccess) e = cudaStreamSynchronize(p->stream);
        if (e != cudaSuccess) return fail_cuda(p, e, "export of the re-keyed records");
        if (vx_write_all(fd, host, n * rb, &written, msg, sizeof msg)) { if (file_bytes) *file_bytes = written; return fail(p, VX_ERR_IO, msg); }
    }
    if (file_bytes) *file_bytes = written;
    return VX_OK;
}

// ------------------------------------------------------------------------------ passes (8(f3))
vx_status vx_plot_passes(const vx_plot *p, uint32_t *passes, uint32_t *selected, uint64_t *bucket_begin,
                         uint64_t *bucket_end)
{
    if (!p) return VX_ERR_ARG;
    if (passes) *passes = 1u << p->g.passes_log;
    if (selected) *selected = p->g.pass;
    if (bucket_begin) *bucket_begin = p->g.b_first;
    if (bucket_end) *bucket_end = p->g.b_first + p->g.NBp;
    return VX_OK;
}

vx_status vx_plot_select_pass(vx_plot *p, uint32_t pass)
{
    if (!p) return VX_ERR_ARG;
    if (pass >= (1u << p->g.passes_log)) return fail(p, VX_ERR_ARG, "pass outside [0, passes)");
    if (p->state >= VX_BUILT) {                            // the workspace is about to be reused
        vx_status s = sync_and_check(p);
        if (s != VX_OK) return s;
    }
    vx_geom_select_pass(&p->g, pass);
    if (p->state > VX_BOUND) p->state = VX_BOUND;          // the tables of the other pass are gone
    p->t1_materialised = false;
    return VX_OK;
}

vx_status vx_plot_all_passes_to_host(vx_plot *p, void *compute_stream, void *copy_stream, uint32_t slices,
                                     void *host_records, size_t records_capacity, uint64_t *host_offsets,
                                     size_t *records_bytes, uint64_t *t1_records)
{
    if (!p) return VX_ERR_ARG;
    if (!host_records) return fail(p, VX_ERR_ARG, "NULL host_records");
    if (p->state < VX_BOUND) return fail(p, VX_ERR_STATE, "vx_plot_all_passes_to_host before vx_plot_bind");
    const uint32_t passes = 1u << p->g.passes_log;
    const size_t rb = p->g.rec2_bytes;
    uint64_t total = 0, t1_total = 0;
    if (records_bytes) *records_bytes = 0;
    for (uint32_t s = 0; s < passes; s++) {
        vx_status st = vx_plot_select_pass(p, s);
        if (st == VX_OK) st = vx_build_table1(p, compute_stream);
        if (st != VX_OK) return st;
        uint64_t n = 0;
        uint64_t *off = host_offsets ? host_offsets + p->g.b_first : NULL;
        st = egress_common(p, compute_stream, copy_stream, slices, (uint8_t *)host_records + total * rb,
                           records_capacity - total * rb, off, NULL, &n);
        if (st != VX_OK) return st;
        if (off && total)                                  // the pass wrote offsets relative to its own first record
            for (uint64_t b = 0; b <= p->g.NBp; b++) off[b] += total;
        uint64_t t1 = 0;
        cudaError_t e = cudaMemcpy(&t1, p->ws + p->g.off_part_base + p->g.P * 8, 8, cudaMemcpyDeviceToHost);
        if (e != cudaSuccess) return fail_cuda(p, e, "cudaMemcpy(part_base)");
        t1_total += t1;
        total += n;
        if (records_bytes) *records_bytes = (size_t)total * rb;
    }
    if (t1_records) *t1_records = t1_total;
    return VX_OK;
}

// ------------------------------------------------------------------------------ one plot over G GPUs (8(f4))
vx_status vx_shard_owner(uint32_t K, uint32_t bucket_bits, uint32_t world, uint32_t rank, uint64_t *nonce_begin,
                         uint64_t *nonce_end, uint64_t *bucket_begin, uint64_t *bucket_end)
{
    if (K < 1 || K > VX_MAX_K || bucket_bits < 1 || bucket_bits > 24) return VX_ERR_ARG;
    if (world < 1 || world > VX_MAX_SHARD_WORLD || (world & (world - 1)) || rank >= world) return VX_ERR_ARG;
    uint32_t wl = 0;
    while ((1u << wl) < world) wl++;
    if (wl > K || wl > bucket_bits) return VX_ERR_ARG;
    if (nonce_begin) *nonce_begin = ((uint64_t)rank << K) >> wl;
    if (nonce_end) *nonce_end = ((uint64_t)(rank + 1) << K) >> wl;
    if (bucket_begin) *bucket_begin = ((uint64_t)rank << bucket_bits) >> wl;
    if (bucket_end) *bucket_end = ((uint64_t)(rank + 1) << bucket_bits) >> wl;
    return VX_OK;
}

static vx_status shard_check(vx_plot *p, uint32_t rank, uint32_t world)
{
    if (p->state < VX_BOUND) return fail(p, VX_ERR_STATE, "sharded build before vx_plot_bind");
    if (world != (1u << p->g.passes_log) || world < 2)
        return fail(p, VX_ERR_ARG, "world must equal the plot's pass count (create with VX_CREATE_PASSES_LOG(log2 world))");
    if (rank >= world) return fail(p, VX_ERR_ARG, "rank outside [0, world)");
    if (p->g.wide) return fail(p, VX_ERR_UNSUPPORTED, "the sharded build is implemented for the 16-byte record layout (K <= 32)");
    return VX_OK;
}

vx_status vx_shard_begin(vx_plot *p, uint32_t rank, uint32_t world, void *cuda_stream)
{
    if (!p) return VX_ERR_ARG;
    vx_status s = shard_check(p, rank, world);
    if (s != VX_OK) return s;
    if (p->state >= VX_BUILT && (s = sync_and_check(p)) != VX_OK && s != VX_ERR_OVERFLOW) return s;
    vx_geom_select_pass(&p->g, rank);                      // the rank owns slice `rank` of the buckets
    p->state = VX_BOUND;
    p->t1_materialised = false;
    p->stream = (cudaStream_t)cuda_stream;
    cudaError_t e = vx_launch_shard_clear(p->g, p->ws, p->stream);
    if (e != cudaSuccess) return fail_cuda(p, e, "shard clear launch");
    return VX_OK;
}

vx_status vx_shard_scatter(vx_plot *p, uint32_t rank, uint32_t world, void *const *dev_peer_workspaces,
                           void *cuda_stream)
{
    if (!p || !dev_peer_workspaces) return VX_ERR_ARG;
    vx_status s = shard_check(p, rank, world);
    if (s != VX_OK) return s;
    if (p->g.pass != rank) return fail(p, VX_ERR_STATE, "vx_shard_scatter before vx_shard_begin for this rank");
    for (uint32_t i = 0; i < world; i++)
        if (!dev_peer_workspaces[i] || ((uintptr_t)dev_peer_workspaces[i] & 255))
            return fail(p, VX_ERR_ARG, "NULL or misaligned peer workspace");
    if (dev_peer_workspaces[rank] != p->ws) return fail(p, VX_ERR_ARG, "peer_workspaces[rank] is not this plot's workspace");
    p->stream = (cudaStream_t)cuda_stream;
    cudaError_t e = vx_launch_shard_scatter(p->g, p->hc, rank, p->g.passes_log, (uint8_t *const *)dev_peer_workspaces, p->stream);
    if (e != cudaSuccess) return fail_cuda(p, e, "shard scatter launch");
    return VX_OK;
}

vx_status vx_shard_finish(vx_plot *p, void *cuda_stream)
{
    if (!p) return VX_ERR_ARG;
    if (p->state < VX_BOUND || !p->g.passes_log) return fail(p, VX_ERR_STATE, "vx_shard_finish before vx_shard_begin");
    p->stream = (cudaStream_t)cuda_stream;
    cudaError_t e = vx_launch_shard_scan(p->g, p->ws, p->stream);
    if (e != cudaSuccess) return fail_cuda(p, e, "shard scan launch");
    p->state = VX_BUILT;
    p->t1_materialised = false;
    return VX_OK;
}

// Peer mapping for ranks that are separate PROCESSES (one per GPU under torch.distributed.run): the
// bound workspace is exported as a CUDA IPC handle of the allocation it lies in plus its offset there
// (PyTorch's caching allocator hands out pieces of larger cudaMalloc blocks), and a peer maps it.
typedef int (*vx_cuMemGetAddressRange_t)(unsigned long long *, size_t *, unsigned long long);

vx_status vx_ipc_export(vx_plot *p, uint8_t handle[64], uint64_t *offset)
{
    if (!p || !handle || !offset) return VX_ERR_ARG;
    if (p->state < VX_BOUND) return fail(p, VX_ERR_STATE, "vx_ipc_export before vx_plot_bind");
    static_assert(sizeof(cudaIpcMemHandle_t) == 64, "CUDA IPC handle size");
    // the base of the allocation: driver API, resolved at run time (libvx does not link libcuda)
    void *drv = dlopen("libcuda.so.1", RTLD_LAZY | RTLD_LOCAL);
    vx_cuMemGetAddressRange_t range = drv ? (vx_cuMemGetAddressRange_t)dlsym(drv, "cuMemGetAddressRange_v2") : NULL;
    if (!range) return fail(p, VX_ERR_CUDA, "libcuda.so.1 / cuMemGetAddressRange_v2 not found");
    unsigned long long base = 0;
    size_t size = 0;
    if (range(&base, &size, (unsigned long long)(uintptr_t)p->ws) != 0)
        return fail(p, VX_ERR_CUDA, "cuMemGetAddressRange failed for the workspace");
    cudaIpcMemHandle_t h;
    cudaError_t e = cudaIpcGetMemHandle(&h, (void *)(uintptr_t)base);
    if (e != cudaSuccess) return fail_cuda(p, e, "cudaIpcGetMemHandle");
    memcpy(handle, &h, 64);
    *offset = (uint64_t)((uintptr_t)p->ws - (uintptr_t)base);
    return VX_OK;
}

vx_status vx_ipc_open(const uint8_t handle[64], uint64_t offset, void **dev_mapped_base, void **dev_workspace)
{
    if (!handle || !dev_mapped_base || !dev_workspace) return VX_ERR_ARG;
    cudaIpcMemHandle_t h;
    memcpy(&h, handle, 64);
    void *base = NULL;
    if (cudaIpcOpenMemHandle(&base, h, cudaIpcMemLazyEnablePeerAccess) != cudaSuccess) {
        cudaGetLastError();
        return VX_ERR_CUDA;
    }
    *dev_mapped_base = base;
    *dev_workspace = (uint8_t *)base + offset;
    return VX_OK;
}

vx_status vx_ipc_close(void *dev_mapped_base)
{
    if (!dev_mapped_base) return VX_ERR_ARG;
    return cudaIpcCloseMemHandle(dev_mapped_base) == cudaSuccess ? VX_OK : VX_ERR_CUDA;
}

vx_status vx_device_tables(vx_plot *p, const void **dev_t1_records, const uint64_t **dev_t1_offsets,
                           const void **dev_t2_records, const uint64_t **dev_t2_offsets,
                           const uint64_t **dev_partition_base)
{
    if (!p) return VX_ERR_ARG;
    if (p->state < VX_MATCHED) return fail(p, VX_ERR_STATE, "vx_device_tables before vx_sort_match_table2");
    if (p->state >= VX_REKEYED) return fail(p, VX_ERR_STATE, "vx_device_tables after vx_rekey_table2 (Table 1 is gone)");
    if (dev_t1_records) *dev_t1_records = p->ws + p->g.off_part;
    if (dev_t1_offsets) *dev_t1_offsets = (const uint64_t *)(p->ws + p->g.off_t1_off);
    if (dev_t2_records) *dev_t2_records = p->ws + p->g.off_t2_rec;
    if (dev_t2_offsets) *dev_t2_offsets = (const uint64_t *)(p->ws + p->g.off_t2_off);
    if (dev_partition_base) *dev_partition_base = (const uint64_t *)(p->ws + p->g.off_part_base);
    return VX_OK;
}

vx_status vx_plot_set_option(vx_plot *p, int option, uint64_t value)
{
    if (!p) return VX_ERR_ARG;
    switch (option) {
    case VX_OPT_FORCE_EXACT_RANK: p->force_exact = value != 0; return VX_OK;
    case VX_OPT_PARTITION_CAPACITY_LIMIT:
        if (value < 1 || value > p->g.cap) return fail(p, VX_ERR_ARG, "limit outside [1, partition capacity]");
        p->g.cap_check = (uint32_t)value;
        return VX_OK;
    case VX_OPT_TABLE2_CAPACITY_LIMIT:
        if (value > p->g.t2_cap) return fail(p, VX_ERR_ARG, "limit above the Table-2 capacity");
        p->g.t2_check = value;
        return VX_OK;
    case VX_OPT_SUBKEY_BITS:
        if (value > 32) return fail(p, VX_ERR_ARG, "sub-key bits outside [0, 32]");
        p->g.subkey_bits = (uint32_t)value;
        return VX_OK;
    case VX_OPT_STAGE2_KERNEL:
        if (value > 1) return fail(p, VX_ERR_ARG, "stage-2 kernel choice outside [0, 1]");
        p->g.s2_kernel = (uint32_t)value;
        return VX_OK;
    }
    return fail(p, VX_ERR_ARG, "unknown option");
}

vx_status vx_get_stats(vx_plot *p, uint64_t *t1_records, uint64_t *t2_records, uint32_t *max_bucket)
{
    if (!p) return VX_ERR_ARG;
    if (p->state < VX_BUILT) return fail(p, VX_ERR_STATE, "vx_get_stats before vx_build_table1");
    vx_status s = sync_and_check(p);
    if (s != VX_OK) return s;
    VxCtrl c;
    cudaError_t e = cudaMemcpy(&c, p->ws + p->g.off_ctrl, sizeof c, cudaMemcpyDeviceToHost);
    if (e != cudaSuccess) return fail_cuda(p, e, "cudaMemcpy(ctrl)");
    uint64_t t1 = 0;
    e = cudaMemcpy(&t1, p->ws + p->g.off_part_base + p->g.P * 8, 8, cudaMemcpyDeviceToHost);
    if (e != cudaSuccess) return fail_cuda(p, e, "cudaMemcpy(part_base)");
    if (t1_records) *t1_records = p->state >= VX_REKEYED ? c.t1_total : t1;
    if (t2_records) *t2_records = p->state >= VX_MATCHED ? c.t2_total : 0;
    if (max_bucket) *max_bucket = p->t1_materialised ? c.max_bucket : 0;
    return VX_OK;
}

vx_status vx_get_counters(vx_plot *p, uint64_t *tile_retries)
{
    if (!p) return VX_ERR_ARG;
    if (p->state < VX_BUILT) return fail(p, VX_ERR_STATE, "vx_get_counters before vx_build_table1");
    vx_status s = sync_and_check(p);
    if (s != VX_OK) return s;
    VxCtrl c;
    cudaError_t e = cudaMemcpy(&c, p->ws + p->g.off_ctrl, sizeof c, cudaMemcpyDeviceToHost);
    if (e != cudaSuccess) return fail_cuda(p, e, "cudaMemcpy(ctrl)");
    if (tile_retries) *tile_retries = c.retries;
    return VX_OK;
}

vx_status vx_hash_range(vx_plot *p, uint64_t nonce_begin, uint64_t count, uint64_t *dev_hashes,
                        void *cuda_stream)
{
    if (!p || (!dev_hashes && count)) return fail(p, VX_ERR_ARG, "NULL argument");
    cudaError_t e = vx_launch_hash_range(p->g, p->hc, nonce_begin, count, dev_hashes, (cudaStream_t)cuda_stream);
    if (e != cudaSuccess) return fail_cuda(p, e, "hash_range launch");
    return VX_OK;
}

vx_status vx_hash_sink(vx_plot *p, uint64_t count, uint64_t *dev_sink, size_t sink_words, void *cuda_stream)
{
    if (!p || !dev_sink) return fail(p, VX_ERR_ARG, "NULL argument");
    cudaError_t e = vx_launch_hash_sink(p->g, p->hc, count, dev_sink, sink_words, (cudaStream_t)cuda_stream);
    if (e != cudaSuccess) return fail_cuda(p, e, "hash_sink launch");
    return VX_OK;
}

vx_status vx_plot_info(const vx_plot *p, uint32_t *K, uint32_t *bucket_bits, uint32_t *nonce_size,
                       uint32_t *partition_bits, uint32_t *partition_capacity, uint64_t *t2_capacity)
{
    if (!p) return VX_ERR_ARG;
    if (K) *K = p->g.K;
    if (bucket_bits) *bucket_bits = p->g.B;
    if (nonce_size) *nonce_size = p->g.nonce_size;
    if (partition_bits) *partition_bits = p->g.pb;
    if (partition_capacity) *partition_capacity = p->g.cap;
    if (t2_capacity) *t2_capacity = p->g.t2_cap;
    return VX_OK;
}

vx_status vx_plot_launches(const vx_plot *p, uint32_t *build_table1, uint32_t *sort_match_table2)
{
    if (!p) return VX_ERR_ARG;
    if (build_table1) *build_table1 = vx_stage1_launches(p->g);
    if (sort_match_table2) *sort_match_table2 = 2;   // clear + the fused kernel
    return VX_OK;
}

vx_status vx_plot_layout(const vx_plot *p, uint32_t *wide, uint32_t *tile_log)
{
    if (!p) return VX_ERR_ARG;
    if (wide) *wide = p->g.wide;
    if (tile_log) *tile_log = p->g.tile_log;
    return VX_OK;
}

const char *vx_last_error(const vx_plot *p) { return p ? p->err : "VX_ERR_ARG: NULL plot"; }

void vx_free(vx_plot *p) { delete p; }

} // extern "C"
