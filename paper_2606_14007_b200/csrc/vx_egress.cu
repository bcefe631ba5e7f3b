// vx_egress.cu -- Table-2 egress pipeline: the fused sort + match stage runs as a
// sequence of partition-range slices, and the Table-2 records and offsets of a finished slice travel
// to the host on a second stream while the later slices are still being sorted and matched.
//
// PAPER.md L81 (III-A): "The completed Table-2 is transferred from VRAM to host over PCIe and
// written to disk in 4 MB sequential chunks"; L91 (III-B): a 256 MB pinned staging buffer; L165/L169
// (the paper's own redo / future-work list): "overlap the PCIe transfer with GPU computation using
// async streams".  The paper's transfer starts after the last kernel; this one starts after the
// first slice.  Two sinks: caller-owned host memory (one copy per slice, straight into place), or a
// file descriptor through a caller-owned pinned ring of 4 MB chunks, written sequentially.
#include <errno.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>
#include <unistd.h>

#include "../../include/vx.h"
#include "vx_internal.h"

#define VX_EGRESS_CHUNK ((size_t)4 << 20)   // 4 MB sequential writes
#define VX_EGRESS_MAX_SLICES 256u
#define VX_EGRESS_PIECE ((uint64_t)1 << 30)  // largest single D2H copy of the memory sink
#define VX_EGRESS_ALIGN ((uint64_t)2 << 20)  // copy boundaries of the memory sink

// Host-mapped mailboxes for the slice ends (the last tile of a slice writes the running |Table 2|
// there).  Allocated once per process and never freed: cudaHostAlloc costs milliseconds and
// cudaFreeHost was seen to block for 0.4 s behind other work, far too much for a per-call buffer.
#include <mutex>
#define VX_MAILBOXES 16
#define VX_MAILBOX_WORDS (VX_EGRESS_MAX_SLICES + 8)   // slice ends + a copy of the control block
static std::mutex g_mb_mutex;
static unsigned long long *g_mb_host = nullptr, *g_mb_dev = nullptr;
static uint32_t g_mb_busy = 0;

static int mailbox_acquire(unsigned long long **host, unsigned long long **dev, cudaError_t *e)
{
    std::lock_guard<std::mutex> lock(g_mb_mutex);
    *e = cudaSuccess;
    if (!g_mb_host) {
        *e = cudaHostAlloc((void **)&g_mb_host, (size_t)VX_MAILBOXES * VX_MAILBOX_WORDS * sizeof(unsigned long long),
                           cudaHostAllocMapped | cudaHostAllocPortable);
        if (*e == cudaSuccess) *e = cudaHostGetDevicePointer((void **)&g_mb_dev, g_mb_host, 0);
        if (*e != cudaSuccess) { if (g_mb_host) cudaFreeHost(g_mb_host); g_mb_host = nullptr; return -1; }
    }
    for (int i = 0; i < VX_MAILBOXES; i++)
        if (!(g_mb_busy & (1u << i))) {
            g_mb_busy |= 1u << i;
            *host = g_mb_host + (size_t)i * VX_MAILBOX_WORDS;
            *dev = g_mb_dev + (size_t)i * VX_MAILBOX_WORDS;
            return i;
        }
    return -1;                                          // *e == cudaSuccess: more than VX_MAILBOXES egress calls in flight
}

static void mailbox_release(int i)
{
    std::lock_guard<std::mutex> lock(g_mb_mutex);
    if (i >= 0) g_mb_busy &= ~(1u << i);
}

// The control block (overflow flags, |Table 2|) goes to the host through the mailbox as well: a
// cudaMemcpy of 32 bytes would queue on the copy engine behind ANOTHER plot's gigabytes of Table 2
// and stall this plot's host thread until they have drained (two plots in flight, bench.py).
__global__ void vx_k_publish_ctrl(const VxCtrl *__restrict__ ctrl, VxCtrl *__restrict__ out) { *out = *ctrl; }

struct VxRing {
    uint8_t *base;        // pinned, caller-owned
    size_t slots;         // ring depth in 4 MB chunks
    cudaEvent_t *ev;      // copy-complete event per slot
    size_t *bytes;        // payload of the chunk in each slot
    size_t head, tail;    // chunks enqueued / chunks written
    int fd;
    uint64_t written;
};

// write() until everything is out: EINTR is retried, a 0-byte write is an error (it would spin);
// *written grows by the bytes that did go out.  Shared by the ring and the trailer (vx_api.cu).
int vx_write_all(int fd, const uint8_t *src, size_t left, uint64_t *written, char *err, size_t errlen)
{
    while (left) {
        const ssize_t w = write(fd, src, left);
        if (w < 0 && errno == EINTR) continue;
        if (w <= 0) {
            snprintf(err, errlen, "write: %s", w < 0 ? strerror(errno) : "wrote 0 bytes");
            return -1;
        }
        src += w; left -= (size_t)w; *written += (uint64_t)w;
    }
    return 0;
}

static int ring_write_oldest(VxRing *r, char *err, size_t errlen)
{
    const size_t slot = r->tail % r->slots;
    cudaError_t e = cudaEventSynchronize(r->ev[slot]);
    if (e != cudaSuccess) { snprintf(err, errlen, "cudaEventSynchronize: %s", cudaGetErrorString(e)); return -1; }
    if (vx_write_all(r->fd, r->base + slot * VX_EGRESS_CHUNK, r->bytes[slot], &r->written, err, errlen)) return -1;
    r->tail++;
    return 0;
}

// device bytes [src, src + bytes) -> the file, through the ring, in order
static int ring_push(VxRing *r, const uint8_t *dev_src, size_t bytes, cudaStream_t copy, char *err, size_t errlen)
{
    while (bytes) {
        if (r->head - r->tail == r->slots && ring_write_oldest(r, err, errlen)) return -1;
        const size_t slot = r->head % r->slots;
        const size_t n = bytes < VX_EGRESS_CHUNK ? bytes : VX_EGRESS_CHUNK;
        cudaError_t e = cudaMemcpyAsync(r->base + slot * VX_EGRESS_CHUNK, dev_src, n, cudaMemcpyDeviceToHost, copy);
        if (e == cudaSuccess) e = cudaEventRecord(r->ev[slot], copy);
        if (e != cudaSuccess) { snprintf(err, errlen, "cudaMemcpyAsync: %s", cudaGetErrorString(e)); return -1; }
        r->bytes[slot] = n;
        r->head++;
        dev_src += n; bytes -= n;
    }
    return 0;
}

// Shared driver.  host_records != NULL: memory sink.  ring != NULL: file sink.
cudaError_t vx_egress_run(const VxGeom &g, uint8_t *ws, bool force_exact, int num_sms, cudaStream_t compute,
                          cudaStream_t copy, uint32_t slices, uint8_t *host_records, size_t records_capacity,
                          uint64_t *host_offsets, VxRing *ring, uint64_t *t2_records, VxCtrl *ctrl_out,
                          int *soft_error, char *err, size_t errlen)
{
    *soft_error = 0;
    if (slices < 1) slices = 1;
    if (slices > VX_EGRESS_MAX_SLICES) slices = VX_EGRESS_MAX_SLICES;
    if (slices > g.P) slices = (uint32_t)g.P;
    unsigned long long *ends = nullptr, *ends_dev = nullptr;
    cudaEvent_t ev[VX_EGRESS_MAX_SLICES];
    uint32_t made = 0;
    cudaError_t e;
    const int mailbox = mailbox_acquire(&ends, &ends_dev, &e);
    if (mailbox < 0) {
        if (e == cudaSuccess) {
            *soft_error = 4;
            snprintf(err, errlen, "more than %d Table-2 egress calls in flight in this process", VX_MAILBOXES);
        }
        return e;
    }
    memset(ends, 0, slices * sizeof(unsigned long long));
    for (; e == cudaSuccess && made < slices; made++)
        e = cudaEventCreateWithFlags(&ev[made], cudaEventDisableTiming);
    // ---- all compute slices are enqueued up front; the host then follows them with the copies
    const uint64_t P = g.P;
    for (uint32_t s = 0; e == cudaSuccess && s < slices; s++) {
        const uint32_t t0 = (uint32_t)(P * s / slices), t1 = (uint32_t)(P * (s + 1) / slices);
        e = vx_launch_stage2(g, ws, true, force_exact, num_sms, compute, t0, t1, ends_dev + s);
        if (e == cudaSuccess) e = cudaEventRecord(ev[s], compute);
    }
    if (e == cudaSuccess) {
        vx_k_publish_ctrl<<<1, 1, 0, compute>>>((const VxCtrl *)(ws + g.off_ctrl), (VxCtrl *)(ends_dev + VX_EGRESS_MAX_SLICES));
        e = cudaGetLastError();
    }
    const uint8_t *t2_dev = ws + g.off_t2_rec;
    const uint8_t *off_dev = ws + g.off_t2_off;
    // 4-byte nonces: Table 2 is resident in the external format and is copied straight out.  5-byte
    // nonces (K = 33): it is resident packed (uint2 + a byte of high bits), so every chunk first goes
    // through vx_k_export_t2 into the workspace's staging area, on the copy stream, chunk by chunk.
    // The staging area is used as two halves: the conversion of chunk k + 1 (on a stream of its own)
    // runs while chunk k is crossing PCIe.
    const bool packed = g.nonce_size > 4;
    const size_t rb = g.rec2_bytes;
    const size_t half = (g.stage_bytes / 2) & ~(size_t)255;
    uint64_t chunk_rec = half / rb;                       // packed: records per staging half,
    if (chunk_rec >= (1u << 20)) chunk_rec &= ~(uint64_t)((1u << 20) - 1);   // a multiple of 2 MB in bytes
    cudaStream_t xs = nullptr;                            // packed: the conversion kernels' stream
    cudaEvent_t exported[2] = {nullptr, nullptr}, drained[2] = {nullptr, nullptr};
    uint64_t chunk_no = 0;
    if (packed && e == cudaSuccess) {
        e = cudaStreamCreateWithFlags(&xs, cudaStreamNonBlocking);
        for (int h = 0; h < 2 && e == cudaSuccess; h++) {
            e = cudaEventCreateWithFlags(&exported[h], cudaEventDisableTiming);
            if (e == cudaSuccess) e = cudaEventCreateWithFlags(&drained[h], cudaEventDisableTiming);
        }
    }
    uint64_t prev = 0, copied = 0;                        // records accounted for / bytes already enqueued
    for (uint32_t s = 0; e == cudaSuccess && s < slices && !*soft_error; s++) {
        e = cudaEventSynchronize(ev[s]);                  // slice s is sorted, matched and emitted
        if (e != cudaSuccess) break;
        const uint64_t cur = ends[s];
        const uint32_t t0 = (uint32_t)(P * s / slices), t1 = (uint32_t)(P * (s + 1) / slices);
        const uint64_t b0 = (uint64_t)t0 << g.fb, b1 = (uint64_t)t1 << g.fb;
        if (cur < prev || cur > g.t2_check) { snprintf(err, errlen, "Table 2 exceeded its capacity"); *soft_error = 2; break; }
        if (host_records && cur * rb > records_capacity) { snprintf(err, errlen, "records_capacity too small"); *soft_error = 1; break; }
        if (packed) {
            // whole staging chunks only, except behind the last slice
            const uint64_t avail = s + 1 == slices ? cur : cur - cur % chunk_rec;
            uint64_t done = copied / rb;
            while (e == cudaSuccess && done < avail && !*soft_error) {
                const uint64_t n = avail - done < chunk_rec ? avail - done : chunk_rec;
                const int h = (int)(chunk_no & 1);
                const size_t so = h ? half : 0;
                if (chunk_no >= 2) e = cudaStreamWaitEvent(xs, drained[h], 0);   // the half is free again
                if (e == cudaSuccess) e = vx_launch_export_t2(g, ws, done, n, xs, so);
                if (e == cudaSuccess) e = cudaEventRecord(exported[h], xs);
                if (e == cudaSuccess) e = cudaStreamWaitEvent(copy, exported[h], 0);
                if (e != cudaSuccess) break;
                if (host_records)
                    e = cudaMemcpyAsync(host_records + done * rb, ws + g.off_stage + so, n * rb, cudaMemcpyDeviceToHost, copy);
                else if (ring_push(ring, ws + g.off_stage + so, n * rb, copy, err, errlen))
                    *soft_error = 3;
                if (e == cudaSuccess) e = cudaEventRecord(drained[h], copy);
                done += n;
                chunk_no++;
            }
            copied = done * rb;
            if (*soft_error) break;
        } else if (host_records) {
            // copies begin and end on 2 MB boundaries of the record stream (the unaligned tail of a slice
            // travels with the next one) and are at most 1 GB long: measured on this box, D2H into a
            // large pinned buffer runs at 55 GB/s that way, 53.5 GB/s with unaligned ends and
            // 52.2 GB/s as one 17 GB copy
            const uint64_t upto = s + 1 == slices ? cur * rb : (cur * rb) & ~(VX_EGRESS_ALIGN - 1);
            for (uint64_t at = copied; e == cudaSuccess && at < upto; at += VX_EGRESS_PIECE) {
                const size_t n = (size_t)(upto - at < VX_EGRESS_PIECE ? upto - at : VX_EGRESS_PIECE);
                e = cudaMemcpyAsync(host_records + at, t2_dev + at, n, cudaMemcpyDeviceToHost, copy);
            }
            if (upto > copied) copied = upto;
        } else if (cur > prev) {
            if (ring_push(ring, t2_dev + prev * rb, (cur - prev) * rb, copy, err, errlen)) { *soft_error = 3; break; }
        }
        if (e == cudaSuccess && host_offsets)
            e = cudaMemcpyAsync(host_offsets + b0, off_dev + b0 * 8, (b1 - b0 + (s + 1 == slices ? 1 : 0)) * 8,
                                cudaMemcpyDeviceToHost, copy);
        prev = cur;
    }
    if (e == cudaSuccess && ring && !*soft_error) {
        // file sink: the CSR offsets follow the records (they are only complete now), same ring
        if (ring_push(ring, off_dev, (g.NBp + 1) * 8, copy, err, errlen)) *soft_error = 3;
        while (!*soft_error && ring->tail < ring->head)
            if (ring_write_oldest(ring, err, errlen)) *soft_error = 3;
    }
    cudaError_t e2 = cudaStreamSynchronize(copy);
    if (e == cudaSuccess) e = e2;
    e2 = cudaStreamSynchronize(compute);
    if (e == cudaSuccess) e = e2;
    if (xs) { cudaStreamSynchronize(xs); cudaStreamDestroy(xs); }
    for (int h = 0; h < 2; h++) { if (exported[h]) cudaEventDestroy(exported[h]); if (drained[h]) cudaEventDestroy(drained[h]); }
    if (t2_records) *t2_records = prev;
    if (ctrl_out) memcpy(ctrl_out, ends + VX_EGRESS_MAX_SLICES, sizeof(VxCtrl));   // valid: compute has drained
    for (uint32_t i = 0; i < made; i++) cudaEventDestroy(ev[i]);
    mailbox_release(mailbox);
    return e;
}

VxRing *vx_ring_create(void *pinned, size_t bytes, int fd)
{
    VxRing *r = (VxRing *)calloc(1, sizeof(VxRing));
    if (!r) return nullptr;
    r->base = (uint8_t *)pinned;
    r->slots = bytes / VX_EGRESS_CHUNK;
    r->fd = fd;
    if (r->slots > 1024) r->slots = 1024;
    if (r->slots >= 2) {
        r->ev = (cudaEvent_t *)calloc(r->slots, sizeof(cudaEvent_t));
        r->bytes = (size_t *)calloc(r->slots, sizeof(size_t));
    }
    bool ok = r->ev && r->bytes;
    for (size_t i = 0; ok && i < r->slots; i++)
        ok = cudaEventCreateWithFlags(&r->ev[i], cudaEventDisableTiming) == cudaSuccess;
    if (!ok) { vx_ring_destroy(r); return nullptr; }
    return r;
}

uint64_t vx_ring_written(const VxRing *r) { return r->written; }

void vx_ring_destroy(VxRing *r)
{
    if (!r) return;
    if (r->ev) for (size_t i = 0; i < r->slots; i++) if (r->ev[i]) cudaEventDestroy(r->ev[i]);
    free(r->ev); free(r->bytes); free(r);
}
