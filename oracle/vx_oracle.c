/*
 * vx_oracle.c -- plain, slow, single-threaded CPU ORACLE for the VaultxGPU plotting hot path.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may call it.  It shares no code, header,
 * table or helper with paper_2606_14007_b200/csrc (the CUDA path) and neither includes the other.
 *
 * What it computes (PAPER.md = /root/reference/PAPER.md, arxiv/paper_2606_14007; readings
 * A1..A18 = SURVEY.md section 8(c), restated in DESIGN.md):
 *
 *   Step 1  key      = 4 x SplitMix64(seed), little-endian           (BASELINE.json configs)
 *   Step 2  H(n)     = first 8 bytes of the BLAKE3 keyed hash of the NONCE_SIZE little-endian
 *                      bytes of n, read as a big-endian u64           (A1-A5)
 *   Step 3  Table 1  = all (n, H(n)), n in [0, 2^K), grouped into 2^B buckets by the hash
 *                      prefix  bucket = H >> (64 - B),  B = 24        (A6-A8)
 *   Step 4  Table 2  = every unordered pair of distinct records of one bucket whose hashes
 *                      differ by less than T = 2^(64-K), written (n_first, n_second) with
 *                      first = the smaller under (H, n)               (A11-A15)
 *   Step 4' the same set by "sort the bucket, scan forward while H_j - H_i < T"
 *                      ("insertion sort by hash value ... then pairwise matching")
 *   Step 5  canonical forms and external record bytes                 (A10, A12, A13)
 *   Step 6  Table 2 re-keyed by the hash of the pair, and the plot file (A19-A21)
 *
 * Everything is integer arithmetic; results are defined bit-exactly.
 *
 * Pins (tests/test_oracle_*.py, all -m "not gpu"): the BLAKE3 routine against the independent
 * `blake3` Python package and against worked values in tests/golden/; SplitMix64 against its
 * published sequence; bucketing against invariants and the Poisson closed form; Step 4 against
 * Step 4' and against an independent numpy brute force and the closed form E|T2|; the slice halves
 * and the digest modes (large-K parity) against the full-table mode and plain-Python restatements.
 * Parity UNPINNED: agreement with the paper's own plot files / the VaultX prover (the paper prints
 * no table contents and VaultX is unpublished).
 */
#define _POSIX_C_SOURCE 199309L   /* clock_gettime for the timing CLI only */
#include <stdint.h>
#include <stddef.h>
#include <stdlib.h>
#include <string.h>
#include <stdio.h>
#include <time.h>

/* ------------------------------------------------------------------ Step 1: SplitMix64 key -- */
/* SURVEY.md 8(c) Step 1 / BASELINE.json "256-bit plot key from SplitMix64(seed=...)". */
static uint64_t splitmix64_next(uint64_t *s)
{
    uint64_t z;
    *s += 0x9E3779B97F4A7C15ULL;
    z = *s;
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
    return z ^ (z >> 31);
}

uint64_t vxo_splitmix64(uint64_t seed, int index)
{ /* the index-th output (0-based) of the generator started at `seed` */
    uint64_t s = seed, r = 0;
    int i;
    for (i = 0; i <= index; i++) r = splitmix64_next(&s);
    return r;
}

void vxo_key_from_seed(uint64_t seed, uint8_t key[32])
{ /* four successive outputs, each serialised little-endian, concatenated */
    uint64_t s = seed;
    int i, j;
    for (i = 0; i < 4; i++) {
        uint64_t w = splitmix64_next(&s);
        for (j = 0; j < 8; j++) key[8 * i + j] = (uint8_t)(w >> (8 * j));
    }
}

/* ------------------------------------------------------------------ Step 2: BLAKE3 keyed hash */
/* BLAKE3 spec (paper ref [4]), section 2: compression function, one chunk of
 * at most one 64-byte block, keyed_hash mode.  Written from the definition; no unrolling. */
static const uint32_t B3_IV[8] = {
    0x6A09E667u, 0xBB67AE85u, 0x3C6EF372u, 0xA54FF53Au,
    0x510E527Fu, 0x9B05688Cu, 0x1F83D9ABu, 0x5BE0CD19u
};
static const int B3_PERM[16] = { 2, 6, 3, 10, 7, 0, 4, 13, 1, 11, 12, 5, 9, 14, 15, 8 };
enum { B3_CHUNK_START = 1, B3_CHUNK_END = 2, B3_ROOT = 8, B3_KEYED_HASH = 16 };

static uint32_t rotr32(uint32_t x, int r) { return (x >> r) | (x << (32 - r)); }

static void b3_g(uint32_t v[16], int a, int b, int c, int d, uint32_t x, uint32_t y)
{
    v[a] = v[a] + v[b] + x;
    v[d] = rotr32(v[d] ^ v[a], 16);
    v[c] = v[c] + v[d];
    v[b] = rotr32(v[b] ^ v[c], 12);
    v[a] = v[a] + v[b] + y;
    v[d] = rotr32(v[d] ^ v[a], 8);
    v[c] = v[c] + v[d];
    v[b] = rotr32(v[b] ^ v[c], 7);
}

static void b3_round(uint32_t v[16], const uint32_t m[16])
{
    b3_g(v, 0, 4, 8, 12, m[0], m[1]);   /* columns */
    b3_g(v, 1, 5, 9, 13, m[2], m[3]);
    b3_g(v, 2, 6, 10, 14, m[4], m[5]);
    b3_g(v, 3, 7, 11, 15, m[6], m[7]);
    b3_g(v, 0, 5, 10, 15, m[8], m[9]);  /* diagonals */
    b3_g(v, 1, 6, 11, 12, m[10], m[11]);
    b3_g(v, 2, 7, 8, 13, m[12], m[13]);
    b3_g(v, 3, 4, 9, 14, m[14], m[15]);
}

/* compress(): 16 output words.  cv = chaining value (here: the key words), block = 16 message
 * words, counter t, block length, domain flags. */
static void b3_compress(const uint32_t cv[8], const uint32_t block[16], uint64_t t,
                        uint32_t block_len, uint32_t flags, uint32_t out[16])
{
    uint32_t v[16], m[16], p[16];
    int i, r;
    for (i = 0; i < 8; i++) v[i] = cv[i];
    for (i = 0; i < 4; i++) v[8 + i] = B3_IV[i];
    v[12] = (uint32_t)t;
    v[13] = (uint32_t)(t >> 32);
    v[14] = block_len;
    v[15] = flags;
    for (i = 0; i < 16; i++) m[i] = block[i];
    for (r = 0; r < 7; r++) {
        b3_round(v, m);
        if (r < 6) { /* permute the message words between rounds */
            for (i = 0; i < 16; i++) p[i] = m[B3_PERM[i]];
            for (i = 0; i < 16; i++) m[i] = p[i];
        }
    }
    for (i = 0; i < 8; i++) {
        out[i] = v[i] ^ v[i + 8];
        out[i + 8] = v[i + 8] ^ cv[i];
    }
}

/* Keyed hash of a message of len <= 64 bytes (a single block of a single chunk, which is also
 * the root): flags = CHUNK_START | CHUNK_END | ROOT | KEYED_HASH, counter 0.  Writes the first
 * outlen <= 64 output bytes.  Returns 0, or -1 on a bad argument. */
int vxo_blake3_keyed(const uint8_t key[32], const uint8_t *msg, size_t len, uint8_t *out, size_t outlen)
{
    uint8_t block[64];
    uint32_t cv[8], m[16], o[16];
    size_t i;
    if (len > 64 || outlen > 64) return -1;
    memset(block, 0, sizeof block);
    if (len) memcpy(block, msg, len);
    for (i = 0; i < 8; i++)
        cv[i] = (uint32_t)key[4 * i] | ((uint32_t)key[4 * i + 1] << 8) |
                ((uint32_t)key[4 * i + 2] << 16) | ((uint32_t)key[4 * i + 3] << 24);
    for (i = 0; i < 16; i++)
        m[i] = (uint32_t)block[4 * i] | ((uint32_t)block[4 * i + 1] << 8) |
               ((uint32_t)block[4 * i + 2] << 16) | ((uint32_t)block[4 * i + 3] << 24);
    b3_compress(cv, m, 0, (uint32_t)len, B3_CHUNK_START | B3_CHUNK_END | B3_ROOT | B3_KEYED_HASH, o);
    for (i = 0; i < outlen; i++) out[i] = (uint8_t)(o[i / 4] >> (8 * (i % 4)));
    return 0;
}

/* A1: NONCE_SIZE = smallest whole number of bytes holding K bits, at least 4. */
int vxo_nonce_size(int K) { return K <= 32 ? 4 : (K + 7) / 8; }

/* H(n): "converts its global ID to a little-endian nonce, computes a Blake3 keyed
 * hash"; A2 (exactly NONCE_SIZE bytes hashed), A4/A5 (first 8 output bytes, big-endian number). */
uint64_t vxo_hash_nonce(const uint8_t key[32], uint64_t n, int nonce_size)
{
    uint8_t nb[8], hb[8];
    uint64_t H = 0;
    int i;
    for (i = 0; i < nonce_size; i++) nb[i] = (uint8_t)(n >> (8 * i));
    vxo_blake3_keyed(key, nb, (size_t)nonce_size, hb, 8);
    for (i = 0; i < 8; i++) H = (H << 8) | hb[i];
    return H;
}

/* hash a contiguous nonce range into out[0 .. count) */
void vxo_hash_range(const uint8_t key[32], int nonce_size, uint64_t n_begin, uint64_t count, uint64_t *out)
{
    uint64_t i;
    for (i = 0; i < count; i++) out[i] = vxo_hash_nonce(key, n_begin + i, nonce_size);
}

/* ------------------------------------------------------------------ Step 3: Table 1 --------- */
typedef struct { uint64_t H, n; } rec_t;

static int rec_cmp(const void *pa, const void *pb)
{ /* A10: (H ascending, n ascending) */
    const rec_t *a = (const rec_t *)pa, *b = (const rec_t *)pb;
    if (a->H != b->H) return a->H < b->H ? -1 : 1;
    if (a->n != b->n) return a->n < b->n ? -1 : 1;
    return 0;
}

/* Table 1 in canonical form (Step 5): bucket b holds records offsets[b] .. offsets[b+1]-1,
 * each bucket sorted by (H, n).  offsets has 2^B + 1 entries; nonces/hashes have 2^K entries.
 * B = bucket_bits (24 at the paper's settings).  Returns 0, -1 bad args, -2 no memory. */
int vxo_table1(int K, const uint8_t key[32], int bucket_bits,
               uint64_t *offsets, uint64_t *nonces, uint64_t *hashes)
{
    const uint64_t N = 1ULL << K, NB = 1ULL << bucket_bits;
    const int ns = vxo_nonce_size(K);
    uint64_t n, b, *fill;
    rec_t *rec;
    if (K < 1 || K > 40 || bucket_bits < 1 || bucket_bits > 32) return -1;
    rec = (rec_t *)malloc((size_t)N * sizeof *rec);
    fill = (uint64_t *)calloc((size_t)NB, sizeof *fill);
    if (!rec || !fill) { free(rec); free(fill); return -2; }

    /* every nonce is hashed once (Step 2); its bucket is the hash prefix (Step 3, A6) */
    for (b = 0; b <= NB; b++) offsets[b] = 0;
    for (n = 0; n < N; n++) {
        hashes[n] = vxo_hash_nonce(key, n, ns);
        offsets[(hashes[n] >> (64 - bucket_bits)) + 1]++;
    }
    for (b = 0; b < NB; b++) offsets[b + 1] += offsets[b];   /* exact-size buckets (A8) */
    for (n = 0; n < N; n++) {
        b = hashes[n] >> (64 - bucket_bits);
        rec[offsets[b] + fill[b]].H = hashes[n];
        rec[offsets[b] + fill[b]].n = n;
        fill[b]++;
    }
    for (b = 0; b < NB; b++)                                  /* canonical in-bucket order (A10) */
        if (offsets[b + 1] - offsets[b] > 1)
            qsort(rec + offsets[b], (size_t)(offsets[b + 1] - offsets[b]), sizeof *rec, rec_cmp);
    for (n = 0; n < N; n++) { nonces[n] = rec[n].n; hashes[n] = rec[n].H; }
    free(rec); free(fill);
    return 0;
}

/* ------------------------------------------------------------------ Step 4: Table 2 --------- */
typedef struct { uint64_t n1, n2; } pair_t;

static int pair_cmp(const void *pa, const void *pb)
{ /* A13 canonical order inside a bucket: (n1, n2) numerically */
    const pair_t *a = (const pair_t *)pa, *b = (const pair_t *)pb;
    if (a->n1 != b->n1) return a->n1 < b->n1 ? -1 : 1;
    if (a->n2 != b->n2) return a->n2 < b->n2 ? -1 : 1;
    return 0;
}

/* The match threshold (A11): T = 2^(64-K); K >= 1 so T fits in 64 bits. */
static uint64_t match_threshold(int K) { return 1ULL << (64 - K); }

/* Step 4, the DEFINITION: all unordered pairs {r, s}, r != s, of one bucket with |H_r - H_s| < T.
 * The bucket's records are (nonces[i], hashes[i]), i < cnt, in ANY order.  Emits canonical
 * (n1, n2)-sorted pairs into out1/out2 (capacity cap); returns the number of pairs (even if it
 * exceeds cap, in which case only cap were written). */
uint64_t vxo_match_allpairs(int K, uint64_t cnt, const uint64_t *nonces, const uint64_t *hashes,
                            uint64_t *out1, uint64_t *out2, uint64_t cap)
{
    const uint64_t T = match_threshold(K);
    uint64_t r, s, m = 0, kept, i;
    pair_t *tmp = NULL;
    for (r = 0; r < cnt; r++)                       /* count first, so that tmp can be sized */
        for (s = r + 1; s < cnt; s++) {
            uint64_t d = hashes[r] > hashes[s] ? hashes[r] - hashes[s] : hashes[s] - hashes[r];
            if (d < T) m++;
        }
    if (m == 0) return 0;
    tmp = (pair_t *)malloc((size_t)m * sizeof *tmp);
    if (!tmp) return UINT64_MAX;
    m = 0;
    for (r = 0; r < cnt; r++)
        for (s = r + 1; s < cnt; s++) {
            uint64_t d = hashes[r] > hashes[s] ? hashes[r] - hashes[s] : hashes[s] - hashes[r];
            if (d < T) {
                /* first = smaller under (H, n) lexicographic order (A11, A12) */
                int r_first = hashes[r] < hashes[s] || (hashes[r] == hashes[s] && nonces[r] < nonces[s]);
                tmp[m].n1 = r_first ? nonces[r] : nonces[s];
                tmp[m].n2 = r_first ? nonces[s] : nonces[r];
                m++;
            }
        }
    qsort(tmp, (size_t)m, sizeof *tmp, pair_cmp);
    kept = m < cap ? m : cap;
    for (i = 0; i < kept; i++) { out1[i] = tmp[i].n1; out2[i] = tmp[i].n2; }
    free(tmp);
    return m;
}

/* Step 4', the FAST FORM: the bucket must already be sorted by (H, n); for each i scan
 * j = i+1, i+2, ... while H_j - H_i < T.  Same output convention as vxo_match_allpairs. */
uint64_t vxo_match_sorted(int K, uint64_t cnt, const uint64_t *nonces, const uint64_t *hashes,
                          uint64_t *out1, uint64_t *out2, uint64_t cap)
{
    const uint64_t T = match_threshold(K);
    uint64_t i, j, m = 0, kept;
    pair_t *tmp;
    for (i = 0; i < cnt; i++)
        for (j = i + 1; j < cnt && hashes[j] - hashes[i] < T; j++) m++;
    if (m == 0) return 0;
    tmp = (pair_t *)malloc((size_t)m * sizeof *tmp);
    if (!tmp) return UINT64_MAX;
    m = 0;
    for (i = 0; i < cnt; i++)
        for (j = i + 1; j < cnt && hashes[j] - hashes[i] < T; j++) {
            tmp[m].n1 = nonces[i];
            tmp[m].n2 = nonces[j];
            m++;
        }
    qsort(tmp, (size_t)m, sizeof *tmp, pair_cmp);
    kept = m < cap ? m : cap;
    for (i = 0; i < kept; i++) { out1[i] = tmp[i].n1; out2[i] = tmp[i].n2; }
    free(tmp);
    return m;
}

/* Table 2 for a bucket range [b_begin, b_end) of a canonical Table 1.
 * mode 0 = Step 4 (all pairs), mode 1 = Step 4' (sorted scan).
 * t2_offsets gets (b_end - b_begin + 1) entries relative to the first bucket of the range.
 * n1/n2 may be NULL (count only).  Returns the number of Table-2 records, UINT64_MAX on error
 * (capacity too small or out of memory). */
uint64_t vxo_table2(int K, int mode, uint64_t b_begin, uint64_t b_end,
                    const uint64_t *t1_offsets, const uint64_t *nonces, const uint64_t *hashes,
                    uint64_t *t2_offsets, uint64_t *n1, uint64_t *n2, uint64_t cap)
{
    uint64_t b, total = 0;
    for (b = b_begin; b < b_end; b++) {
        const uint64_t o = t1_offsets[b], c = t1_offsets[b + 1] - o;
        const uint64_t room = (n1 && total < cap) ? cap - total : 0;
        uint64_t m;
        if (t2_offsets) t2_offsets[b - b_begin] = total;
        m = mode == 0
          ? vxo_match_allpairs(K, c, nonces + o, hashes + o, n1 ? n1 + total : NULL, n2 ? n2 + total : NULL, room)
          : vxo_match_sorted(K, c, nonces + o, hashes + o, n1 ? n1 + total : NULL, n2 ? n2 + total : NULL, room);
        if (m == UINT64_MAX) return UINT64_MAX;
        if (n1 && m > room) return UINT64_MAX;
        total += m;
    }
    if (t2_offsets) t2_offsets[b_end - b_begin] = total;
    return total;
}

/* ------------------------------------------------------------------ Step 5: external bytes -- */
/* Table-1 record = nonce[NONCE_SIZE] little-endian || the 8 hash bytes (= H big-endian);
 * Table-2 record = nonce1[NONCE_SIZE] || nonce2[NONCE_SIZE], both little-endian (A1, A4, A12). */
void vxo_serialize_t1(int nonce_size, uint64_t cnt, const uint64_t *nonces, const uint64_t *hashes, uint8_t *out)
{
    uint64_t i;
    int j;
    for (i = 0; i < cnt; i++) {
        uint8_t *r = out + i * (uint64_t)(nonce_size + 8);
        for (j = 0; j < nonce_size; j++) r[j] = (uint8_t)(nonces[i] >> (8 * j));
        for (j = 0; j < 8; j++) r[nonce_size + j] = (uint8_t)(hashes[i] >> (8 * (7 - j)));
    }
}

void vxo_serialize_t2(int nonce_size, uint64_t cnt, const uint64_t *n1, const uint64_t *n2, uint8_t *out)
{
    uint64_t i;
    int j;
    for (i = 0; i < cnt; i++) {
        uint8_t *r = out + i * (uint64_t)(2 * nonce_size);
        for (j = 0; j < nonce_size; j++) r[j] = (uint8_t)(n1[i] >> (8 * j));
        for (j = 0; j < nonce_size; j++) r[nonce_size + j] = (uint8_t)(n2[i] >> (8 * j));
    }
}

/* ------------------------------------------------------------------ streaming digests ------- */
/* Large-K parity (SURVEY.md 8(c) "Large-K parity"): order-independent per-bucket digests that a
 * test can recompute from vx_read_tables output with numpy.  f = the SplitMix64 finaliser.
 *   D1[b] = sum over records of bucket b of f(H ^ f(n))            (mod 2^64)
 *   D2[b] = sum over Table-2 records of bucket b of f(f(n1) ^ n2)  (mod 2^64) */
static uint64_t mix64(uint64_t z)
{
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
    return z ^ (z >> 31);
}
uint64_t vxo_mix64(uint64_t z) { return mix64(z); }

/* Slice mode for K too large to hold on the host, in two halves so that several single-threaded
 * workers can share the hashing (SURVEY.md 8(c) "Large-K parity": "run the slices as independent
 * single-threaded processes on separate cores"):
 *   vxo_filter_range        hashes the nonces [n_begin, n_end) and keeps, in nonce order, the records
 *                           whose bucket lies in [b_begin, b_end)               (Steps 2 and 3)
 *   vxo_table1_from_records puts records given in ANY order into the canonical form of vxo_table1 for
 *                           that bucket range: offsets relative to b_begin, buckets sorted by (H, n)
 * vxo_table1_slice is the one after the other over all 2^K nonces. */
uint64_t vxo_filter_range(const uint8_t key[32], int nonce_size, int bucket_bits, uint64_t b_begin, uint64_t b_end,
                          uint64_t n_begin, uint64_t n_end, uint64_t *nonces, uint64_t *hashes, uint64_t cap)
{ /* returns the number of records kept, or UINT64_MAX if cap is too small */
    uint64_t n, kept = 0;
    for (n = n_begin; n < n_end; n++) {
        const uint64_t H = vxo_hash_nonce(key, n, nonce_size);
        const uint64_t b = H >> (64 - bucket_bits);
        if (b < b_begin || b >= b_end) continue;
        if (kept == cap) return UINT64_MAX;
        nonces[kept] = n; hashes[kept] = H; kept++;
    }
    return kept;
}

int vxo_table1_from_records(int bucket_bits, uint64_t b_begin, uint64_t b_end, uint64_t cnt,
                            const uint64_t *nonces_in, const uint64_t *hashes_in,
                            uint64_t *offsets, uint64_t *nonces, uint64_t *hashes)
{ /* 0, -1 a record outside the bucket range, -2 no memory */
    const uint64_t nb = b_end - b_begin;
    uint64_t i, b, *fill;
    rec_t *rec;
    rec = (rec_t *)malloc((size_t)(cnt ? cnt : 1) * sizeof *rec);
    fill = (uint64_t *)calloc((size_t)(nb ? nb : 1), sizeof *fill);
    if (!rec || !fill) { free(rec); free(fill); return -2; }
    for (b = 0; b <= nb; b++) offsets[b] = 0;
    for (i = 0; i < cnt; i++) {
        b = hashes_in[i] >> (64 - bucket_bits);
        if (b < b_begin || b >= b_end) { free(rec); free(fill); return -1; }
        offsets[b - b_begin + 1]++;
    }
    for (b = 0; b < nb; b++) offsets[b + 1] += offsets[b];   /* exact-size buckets (A8) */
    for (i = 0; i < cnt; i++) {
        b = (hashes_in[i] >> (64 - bucket_bits)) - b_begin;
        rec[offsets[b] + fill[b]].H = hashes_in[i];
        rec[offsets[b] + fill[b]].n = nonces_in[i];
        fill[b]++;
    }
    for (b = 0; b < nb; b++)                                  /* canonical in-bucket order (A10) */
        if (offsets[b + 1] - offsets[b] > 1)
            qsort(rec + offsets[b], (size_t)(offsets[b + 1] - offsets[b]), sizeof *rec, rec_cmp);
    for (i = 0; i < cnt; i++) { nonces[i] = rec[i].n; hashes[i] = rec[i].H; }
    free(rec); free(fill);
    return 0;
}

/* hashes ALL 2^K nonces but keeps only the records whose bucket lies in [b_begin, b_end); returns
 * them canonically (as vxo_table1 does for the whole table) with offsets relative to b_begin.
 * cap = capacity of nonces/hashes.  Returns the number of records kept, or UINT64_MAX if cap is
 * too small / out of memory. */
uint64_t vxo_table1_slice(int K, const uint8_t key[32], int bucket_bits, uint64_t b_begin, uint64_t b_end,
                          uint64_t *offsets, uint64_t *nonces, uint64_t *hashes, uint64_t cap)
{
    uint64_t kept, *rn, *rh;
    rn = (uint64_t *)malloc((size_t)(cap ? cap : 1) * sizeof *rn);
    rh = (uint64_t *)malloc((size_t)(cap ? cap : 1) * sizeof *rh);
    if (!rn || !rh) { free(rn); free(rh); return UINT64_MAX; }
    kept = vxo_filter_range(key, vxo_nonce_size(K), bucket_bits, b_begin, b_end, 0, 1ULL << K, rn, rh, cap);
    if (kept != UINT64_MAX && vxo_table1_from_records(bucket_bits, b_begin, b_end, kept, rn, rh, offsets, nonces, hashes) != 0)
        kept = UINT64_MAX;
    free(rn); free(rh);
    return kept;
}

/* Digest mode: one pass over all nonces keeping only count1[b] and D1[b] for every bucket
 * (2 x 2^B u64 of host memory).  Used to check every bucket of a large-K GPU Table 1. */
int vxo_table1_digest(int K, const uint8_t key[32], int bucket_bits, uint64_t *count1, uint64_t *D1)
{
    const uint64_t N = 1ULL << K, NB = 1ULL << bucket_bits;
    const int ns = vxo_nonce_size(K);
    uint64_t n, b;
    if (K < 1 || K > 40 || bucket_bits < 1 || bucket_bits > 32) return -1;
    for (b = 0; b < NB; b++) { count1[b] = 0; D1[b] = 0; }
    for (n = 0; n < N; n++) {
        const uint64_t H = vxo_hash_nonce(key, n, ns);
        b = H >> (64 - bucket_bits);
        count1[b]++;
        D1[b] += mix64(H ^ mix64(n));
    }
    return 0;
}

/* Table-2 digest mode: count2[b] and D2[b] (above) for the buckets [b_begin, b_end) of a canonical
 * Table 1, entries relative to b_begin.  Bucket by bucket it is Step 4 (mode 0) or Step 4' (mode 1)
 * exactly as vxo_table2 runs them; only the records are folded into the digest instead of being kept.
 * Returns the number of Table-2 records, UINT64_MAX if out of memory. */
uint64_t vxo_table2_digest(int K, int mode, uint64_t b_begin, uint64_t b_end,
                           const uint64_t *t1_offsets, const uint64_t *nonces, const uint64_t *hashes,
                           uint64_t *count2, uint64_t *D2)
{
    uint64_t b, total = 0;
    for (b = b_begin; b < b_end; b++) {
        const uint64_t o = t1_offsets[b], c = t1_offsets[b + 1] - o;
        uint64_t m, i, d = 0, *p1 = NULL, *p2 = NULL;
        m = mode == 0 ? vxo_match_allpairs(K, c, nonces + o, hashes + o, NULL, NULL, 0)
                      : vxo_match_sorted(K, c, nonces + o, hashes + o, NULL, NULL, 0);
        if (m == UINT64_MAX) return UINT64_MAX;
        if (m) {
            p1 = (uint64_t *)malloc((size_t)m * sizeof *p1);
            p2 = (uint64_t *)malloc((size_t)m * sizeof *p2);
            if (!p1 || !p2) { free(p1); free(p2); return UINT64_MAX; }
            if (mode == 0) vxo_match_allpairs(K, c, nonces + o, hashes + o, p1, p2, m);
            else vxo_match_sorted(K, c, nonces + o, hashes + o, p1, p2, m);
            for (i = 0; i < m; i++) d += mix64(mix64(p1[i]) ^ p2[i]);
            free(p1); free(p2);
        }
        count2[b - b_begin] = m;
        D2[b - b_begin] = d;
        total += m;
    }
    return total;
}

/* ------------------------------------------------------------------ Step 6: re-keyed Table 2 */
/* SURVEY.md 8(f2) (plot files a prover searches): Table 2 comes out of the
 * match step grouped by the bucket of the TABLE-1 hash, so nothing can look a challenge up in it.
 * The paper does not say how VaultX keys it (the format is unpublished, L183); readings A19-A21 of
 * DESIGN.md fix this build's own:
 *   A19  pair hash  H2(n1, n2) = first 8 bytes, read big-endian, of the BLAKE3 keyed hash (same plot
 *        key, same mode as Step 2) of the external Table-2 record bytes
 *        nonce1[NONCE_SIZE] LE || nonce2[NONCE_SIZE] LE   (block_len = 2 NONCE_SIZE);
 *   A20  the re-keyed table holds the same pairs, grouped into 2^B buckets by H2 >> (64 - B), each
 *        bucket sorted by (H2, n1, n2); CSR offsets;
 *   A21  plot file = header || offsets || records (vxo_plot_file below).
 * Parity with VaultX's own files: UNPINNED (as for Table 2 itself). */
uint64_t vxo_hash_pair(const uint8_t key[32], uint64_t n1, uint64_t n2, int nonce_size)
{
    uint8_t msg[16], hb[8];
    uint64_t H = 0;
    int i;
    for (i = 0; i < nonce_size; i++) msg[i] = (uint8_t)(n1 >> (8 * i));
    for (i = 0; i < nonce_size; i++) msg[nonce_size + i] = (uint8_t)(n2 >> (8 * i));
    vxo_blake3_keyed(key, msg, (size_t)(2 * nonce_size), hb, 8);
    for (i = 0; i < 8; i++) H = (H << 8) | hb[i];
    return H;
}

typedef struct { uint64_t H, n1, n2; } rk_t;

static int rk_cmp(const void *pa, const void *pb)
{ /* A20: (H2, n1, n2) ascending */
    const rk_t *a = (const rk_t *)pa, *b = (const rk_t *)pb;
    if (a->H != b->H) return a->H < b->H ? -1 : 1;
    if (a->n1 != b->n1) return a->n1 < b->n1 ? -1 : 1;
    if (a->n2 != b->n2) return a->n2 < b->n2 ? -1 : 1;
    return 0;
}

/* cnt pairs (n1[i], n2[i]) in any order -> offsets[2^B + 1], and the pairs with their hashes in the
 * canonical order of A20.  Returns 0, -1 bad args, -2 no memory. */
int vxo_table2_rekey(int K, const uint8_t key[32], int bucket_bits, uint64_t cnt,
                     const uint64_t *n1, const uint64_t *n2,
                     uint64_t *offsets, uint64_t *n1_out, uint64_t *n2_out, uint64_t *h2_out)
{
    const uint64_t NB = 1ULL << bucket_bits;
    const int ns = vxo_nonce_size(K);
    uint64_t i, b, *fill;
    rk_t *rec, *tmp;
    if (K < 1 || K > 40 || bucket_bits < 1 || bucket_bits > 32) return -1;
    rec = (rk_t *)malloc((size_t)(cnt ? cnt : 1) * sizeof *rec);
    tmp = (rk_t *)malloc((size_t)(cnt ? cnt : 1) * sizeof *tmp);
    fill = (uint64_t *)calloc((size_t)NB, sizeof *fill);
    if (!rec || !tmp || !fill) { free(rec); free(tmp); free(fill); return -2; }
    for (b = 0; b <= NB; b++) offsets[b] = 0;
    for (i = 0; i < cnt; i++) {
        tmp[i].H = vxo_hash_pair(key, n1[i], n2[i], ns);
        tmp[i].n1 = n1[i]; tmp[i].n2 = n2[i];
        offsets[(tmp[i].H >> (64 - bucket_bits)) + 1]++;
    }
    for (b = 0; b < NB; b++) offsets[b + 1] += offsets[b];
    for (i = 0; i < cnt; i++) {
        b = tmp[i].H >> (64 - bucket_bits);
        rec[offsets[b] + fill[b]++] = tmp[i];
    }
    for (b = 0; b < NB; b++)
        if (offsets[b + 1] - offsets[b] > 1)
            qsort(rec + offsets[b], (size_t)(offsets[b + 1] - offsets[b]), sizeof *rec, rk_cmp);
    for (i = 0; i < cnt; i++) { n1_out[i] = rec[i].n1; n2_out[i] = rec[i].n2; h2_out[i] = rec[i].H; }
    free(rec); free(tmp); free(fill);
    return 0;
}

/* A21, the plot file: 64-byte header
 *     "VXPLOT" 0x00 0x01 | u32 K | u32 B | u32 NONCE_SIZE | u32 0 | key[32] | u64 record count
 * then (2^B + 1) u64 CSR offsets (in records), then the records nonce1[NONCE_SIZE] || nonce2[NONCE_SIZE]
 * bucket-major; all integers little-endian.  Writes into out (size vxo_plot_file_bytes). */
uint64_t vxo_plot_file_bytes(int K, int bucket_bits, uint64_t cnt)
{
    return 64 + 8 * ((1ULL << bucket_bits) + 1) + cnt * (uint64_t)(2 * vxo_nonce_size(K));
}

void vxo_plot_file(int K, const uint8_t key[32], int bucket_bits, uint64_t cnt, const uint64_t *offsets,
                   const uint64_t *n1, const uint64_t *n2, uint8_t *out)
{
    const uint64_t NB = 1ULL << bucket_bits;
    const int ns = vxo_nonce_size(K);
    const uint32_t w[4] = { (uint32_t)K, (uint32_t)bucket_bits, (uint32_t)ns, 0u };
    uint64_t b;
    int i, j;
    memcpy(out, "VXPLOT\0\1", 8);
    for (i = 0; i < 4; i++) for (j = 0; j < 4; j++) out[8 + 4 * i + j] = (uint8_t)(w[i] >> (8 * j));
    memcpy(out + 24, key, 32);
    for (j = 0; j < 8; j++) out[56 + j] = (uint8_t)(cnt >> (8 * j));
    for (b = 0; b <= NB; b++) for (j = 0; j < 8; j++) out[64 + 8 * b + j] = (uint8_t)(offsets[b] >> (8 * j));
    vxo_serialize_t2(ns, cnt, n1, n2, out + 64 + 8 * (NB + 1));
}

/* ------------------------------------------------------------------ tiny CLI / timing ------- */
#ifdef VXO_MAIN
static double now_s(void)
{
    struct timespec ts;
    clock_gettime(CLOCK_MONOTONIC, &ts);
    return (double)ts.tv_sec + 1e-9 * (double)ts.tv_nsec;
}

int main(int argc, char **argv)
{
    int K = argc > 1 ? atoi(argv[1]) : 16, B = argc > 3 ? atoi(argv[3]) : 24;
    uint64_t seed = argc > 2 ? strtoull(argv[2], NULL, 0) : 1, N, NB, total;
    uint8_t key[32];
    uint64_t *off, *non, *has;
    double t0, t1, t2;
    int i;
    if (K < 1 || K > 32 || B < 1 || B > 28) { fprintf(stderr, "usage: vx_oracle K seed [B]\n"); return 2; }
    N = 1ULL << K; NB = 1ULL << B;
    vxo_key_from_seed(seed, key);
    printf("K=%d seed=%llu B=%d key=", K, (unsigned long long)seed, B);
    for (i = 0; i < 32; i++) printf("%02x", key[i]);
    printf("\n");
    off = (uint64_t *)malloc((size_t)(NB + 1) * 8);
    non = (uint64_t *)malloc((size_t)N * 8);
    has = (uint64_t *)malloc((size_t)N * 8);
    if (!off || !non || !has) return 1;
    t0 = now_s();
    if (vxo_table1(K, key, B, off, non, has)) return 1;
    t1 = now_s();
    total = vxo_table2(K, 1, 0, NB, off, non, has, NULL, NULL, NULL, 0);
    t2 = now_s();
    printf("table1: %llu records in %.3f s (%.3f M nonces/s)\n", (unsigned long long)N, t1 - t0, N / (t1 - t0) / 1e6);
    printf("table2: %llu records in %.3f s\n", (unsigned long long)total, t2 - t1);
    free(off); free(non); free(has);
    return 0;
}
#endif
