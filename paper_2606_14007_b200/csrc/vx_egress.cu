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

struct VxRing {
    uint8_t *base;        // pinned, caller-owned
    size_t slots;         // ring depth in 4 MB chunks
    cudaEvent_t *ev;      // copy-complete event per slot
    size_t *bytes;        // payload of the chunk in each slot
    size_t head, tail;    // chunks enqueued / chunks written
    int fd;
    uint64_t written;
};

static int ring_write_oldest(VxRing *r, char *err, size_t errlen)
{
    const size_t slot = r->tail % r->slots;
    cudaError_t e = cudaEventSynchronize(r->ev[slot]);
    if (e != cudaSuccess) { snprintf(err, errlen, "cudaEventSynchronize: %s", cudaGetErrorString(e)); return -1; }
    const uint8_t *src = r->base + slot * VX_EGRESS_CHUNK;
    size_t left = r->bytes[slot];
    while (left) {
        const ssize_t w = write(r->fd, src, left);
        if (w < 0) {
            if (errno == EINTR) continue;
            snprintf(err, errlen, "write: %s", strerror(errno));
            return -1;
        }
        src += w; left -= (size_t)w; r->written += (uint64_t)w;
    }
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
                          uint64_t *host_offsets, VxRing *ring, uint64_t *t2_records, int *soft_error,
                          char *err, size_t errlen)
{
    *soft_error = 0;
    if (slices < 1) slices = 1;
    if (slices > VX_EGRESS_MAX_SLICES) slices = VX_EGRESS_MAX_SLICES;
    if (slices > g.P) slices = (uint32_t)g.P;
    unsigned long long *ends = nullptr, *ends_dev = nullptr;
    cudaEvent_t ev[VX_EGRESS_MAX_SLICES];
    uint32_t made = 0;
    cudaError_t e = cudaHostAlloc((void **)&ends, slices * sizeof(unsigned long long), cudaHostAllocMapped);
    if (e != cudaSuccess) return e;
    memset(ends, 0, slices * sizeof(unsigned long long));
    e = cudaHostGetDevicePointer((void **)&ends_dev, ends, 0);
    for (; e == cudaSuccess && made < slices; made++)
        e = cudaEventCreateWithFlags(&ev[made], cudaEventDisableTiming);
    // ---- all compute slices are enqueued up front; the host then follows them with the copies
    const uint64_t P = g.P;
    for (uint32_t s = 0; e == cudaSuccess && s < slices; s++) {
        const uint32_t t0 = (uint32_t)(P * s / slices), t1 = (uint32_t)(P * (s + 1) / slices);
        e = vx_launch_stage2(g, ws, true, force_exact, num_sms, compute, t0, t1, ends_dev + s);
        if (e == cudaSuccess) e = cudaEventRecord(ev[s], compute);
    }
    const uint8_t *t2_dev = ws + g.off_t2_rec;
    const uint8_t *off_dev = ws + g.off_t2_off;
    const size_t rb = 8;                                  // narrow Table-2 records are resident in the external format
    uint64_t prev = 0;
    for (uint32_t s = 0; e == cudaSuccess && s < slices && !*soft_error; s++) {
        e = cudaEventSynchronize(ev[s]);                  // slice s is sorted, matched and emitted
        if (e != cudaSuccess) break;
        const uint64_t cur = ends[s];
        const uint32_t t0 = (uint32_t)(P * s / slices), t1 = (uint32_t)(P * (s + 1) / slices);
        const uint64_t b0 = (uint64_t)t0 << g.fb, b1 = (uint64_t)t1 << g.fb;
        if (cur < prev || cur > g.t2_check) { snprintf(err, errlen, "Table 2 exceeded its capacity"); *soft_error = 2; break; }
        if (host_records) {
            if (cur * rb > records_capacity) { snprintf(err, errlen, "records_capacity too small"); *soft_error = 1; break; }
            if (cur > prev)
                e = cudaMemcpyAsync(host_records + prev * rb, t2_dev + prev * rb, (cur - prev) * rb, cudaMemcpyDeviceToHost, copy);
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
        if (ring_push(ring, off_dev, (g.NB + 1) * 8, copy, err, errlen)) *soft_error = 3;
        while (!*soft_error && ring->tail < ring->head)
            if (ring_write_oldest(ring, err, errlen)) *soft_error = 3;
    }
    cudaError_t e2 = cudaStreamSynchronize(copy);
    if (e == cudaSuccess) e = e2;
    e2 = cudaStreamSynchronize(compute);
    if (e == cudaSuccess) e = e2;
    if (t2_records) *t2_records = prev;
    for (uint32_t i = 0; i < made; i++) cudaEventDestroy(ev[i]);
    cudaFreeHost(ends);
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
