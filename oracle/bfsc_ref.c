/*
 * bfsc_ref.c — the ORACLE (test infrastructure; see bfsc_ref.h for scope, citations, pins).
 * Plain scalar C, no SIMD, no blocking or fusion beyond what FORMAT.md states.
 * Step labels O1..O7 are SURVEY.md §8(c)'s; "L<n>" are lines of /root/reference/PAPER.md.
 */
#include "bfsc_ref.h"

#include <pthread.h>
#include <stdlib.h>
#include <string.h>

#define BLK 128

static size_t align_up(size_t x, size_t k) { return (x + k - 1) / k * k; }

/* ---- little-endian stores/loads, byte by byte (host-endianness independent) ---- */
static void st_le(uint8_t *p, uint64_t v, int nbytes) {
    for (int i = 0; i < nbytes; i++) p[i] = (uint8_t)(v >> (8 * i));
}
static uint64_t ld_le(const uint8_t *p, int nbytes) {
    uint64_t v = 0;
    for (int i = 0; i < nbytes; i++) v |= (uint64_t)p[i] << (8 * i);
    return v;
}
static uint64_t load_id(const void *ids, size_t i, int W) {
    return W == 32 ? (uint64_t)((const uint32_t *)ids)[i] : ((const uint64_t *)ids)[i];
}
static void store_id(void *ids, size_t i, int W, uint64_t v) {
    if (W == 32) ((uint32_t *)ids)[i] = (uint32_t)v; else ((uint64_t *)ids)[i] = v;
}
static uint64_t wmask(int W) { return W == 64 ? ~(uint64_t)0 : (((uint64_t)1 << W) - 1); }

/* eq. (6): size = ceil(log2(max+1-min)) = bit length of (max-min). */
int bfsc_ref_width(uint64_t v) {
    int w = 0;
    while (v) { w++; v >>= 1; }
    return w;
}

size_t bfsc_ref_block_bytes(int b, int n_exc, int W) {
    size_t s = 16 + 16 * (size_t)b;
    if (n_exc > 0) s += align_up(align_up((size_t)n_exc, (size_t)W / 8) + (size_t)n_exc * (size_t)(W / 8), 16);
    return s;
}

static size_t n_blocks(size_t n) { return (n + BLK - 1) / BLK; }
static size_t dir_bytes(size_t nb) { return align_up(4 * (nb + 1), 16); }

size_t bfsc_ref_compress_bound(size_t n, int W) {
    size_t nb = n_blocks(n);
    return 32 + dir_bytes(nb) + nb * (16 + 16 * (size_t)W);
}

/* O3: delta coding (L979-986), modular, base = first ID of the block, zero padded. */
uint64_t bfsc_ref_block_deltas(const void *x, int m, int W, uint64_t d[128]) {
    uint64_t mask = wmask(W);
    uint64_t base = load_id(x, 0, W);
    d[0] = 0;
    for (int j = 1; j < m; j++) d[j] = (load_id(x, (size_t)j, W) - load_id(x, (size_t)j - 1, W)) & mask;
    for (int j = m; j < BLK; j++) d[j] = 0;
    return base;
}

/* O4 + O5: widths, exception counts, argmin of the exact block size, ties -> largest b. */
int bfsc_ref_choose_b(const uint64_t d[128], int W, int *n_exc_out) {
    int w[BLK], maxw = 0;
    for (int j = 0; j < BLK; j++) { w[j] = bfsc_ref_width(d[j]); if (w[j] > maxw) maxw = w[j]; }
    int best_b = 0, best_exc = 0; size_t best_size = (size_t)-1;
    for (int b = 0; b <= maxw; b++) {
        int n_exc = 0;
        for (int j = 0; j < BLK; j++) if (w[j] > b) n_exc++;       /* d_j >= 2^b, L1011 */
        size_t s = bfsc_ref_block_bytes(b, n_exc, W);
        if (s <= best_size) { best_size = s; best_b = b; best_exc = n_exc; }  /* <= : tie -> larger b */
    }
    if (n_exc_out) *n_exc_out = best_exc;
    return best_b;
}

/* FORMAT.md §7 (mode 2, BP128-D1): plain binary packing, the codec class the thesis ran (S4-BP128,
 * blocks of 128, b in 0..32, no exceptions). b = the frame-of-reference width of
 * the block's deltas (eq. 6 L969 with min = 0; "driven by b of the worst value", L987-998). */
int bfsc_ref_choose_b_bp128(const uint64_t d[128]) {
    int maxw = 0;
    for (int j = 0; j < BLK; j++) { int w = bfsc_ref_width(d[j]); if (w > maxw) maxw = w; }
    return maxw;
}

/* O6: header, payload (4-column interleave), exceptions, pads — FORMAT.md §2. */
size_t bfsc_ref_emit_block(const uint64_t d[128], uint64_t base, int b, int W, uint8_t *out) {
    int pos[BLK], n_exc = 0;
    for (int j = 0; j < BLK; j++)
        if (bfsc_ref_width(d[j]) > b) pos[n_exc++] = j;
    size_t size = bfsc_ref_block_bytes(b, n_exc, W);
    memset(out, 0, size);
    st_le(out, base, 8);
    out[8] = (uint8_t)b;
    out[9] = (uint8_t)n_exc;
    uint8_t *payload = out + 16;
    /* value j: column c = j%4, row r = j/4; bit i of its low part -> bit r*b+i of column c's
     * stream; stream bit s lives in 32-bit LE word s/32 at payload byte 16*(s/32) + 4c. */
    for (int j = 0; j < BLK; j++) {
        int c = j % 4, r = j / 4;
        for (int i = 0; i < b; i++) {
            if ((d[j] >> i) & 1) {
                int s = r * b + i;
                int word = s / 32, bit = s % 32;
                payload[16 * word + 4 * c + bit / 8] |= (uint8_t)(1u << (bit % 8));
            }
        }
    }
    if (n_exc > 0) {
        uint8_t *e = payload + 16 * (size_t)b;
        for (int i = 0; i < n_exc; i++) e[i] = (uint8_t)pos[i];
        uint8_t *h = e + align_up((size_t)n_exc, (size_t)W / 8);
        for (int i = 0; i < n_exc; i++) {
            uint64_t high = (b >= 64) ? 0 : (d[pos[i]] >> b);   /* b == W never has exceptions */
            st_le(h + (size_t)i * (W / 8), high, W / 8);
        }
    }
    return size;
}

static void write_header(uint8_t *out, int W, int mode, uint64_t n, uint64_t total, uint32_t nb) {
    memset(out, 0, 32);
    out[0] = 'B'; out[1] = 'F'; out[2] = 'S'; out[3] = 'C';
    out[4] = 1; out[5] = (uint8_t)W; out[6] = (uint8_t)mode;
    st_le(out + 8, n, 8);
    st_le(out + 16, total, 8);
    st_le(out + 24, nb, 4);
}

/* O1: RAW iff n*W/8 < threshold (L1311: minimum size that triggers compression). */
static int is_raw(size_t n, int W, size_t thr) { return n * (size_t)(W / 8) < thr; }

int bfsc_ref_compress(const void *ids, size_t n, int W, size_t thr,
                      uint8_t *out, size_t cap, size_t *out_bytes) {
    return bfsc_ref_compress_codec(BFSC_REF_CODEC_PFOR, ids, n, W, thr, out, cap, out_bytes);
}

static int compress_rule(int codec, const void *ids, size_t n, int W, size_t thr,
                         uint8_t *out, size_t cap, size_t *out_bytes);

/* FORMAT.md §8: with BFSC_REF_FLAG_RAW_FALLBACK the stream is encoded under the rule, and sent RAW after all when that
 * did not make it smaller than the RAW stream of the same IDs ("Compression -> Transmission -> Decompression slower
 * than Transmission"; the thesis sets its threshold by hand, L2086, L2164). Written the plain way:
 * encode, compare, encode again as RAW. */
int bfsc_ref_compress_codec(int codec, const void *ids, size_t n, int W, size_t thr,
                            uint8_t *out, size_t cap, size_t *out_bytes) {
    int fallback = codec & BFSC_REF_FLAG_RAW_FALLBACK;
    codec &= ~BFSC_REF_FLAG_RAW_FALLBACK;
    int rc = compress_rule(codec, ids, n, W, thr, out, cap, out_bytes);
    if (rc || !fallback) return rc;
    size_t raw_total = 32 + align_up(n * (size_t)(W / 8), 16);
    if (*out_bytes >= raw_total)                               /* did not shrink: RAW (threshold above any size) */
        return compress_rule(codec, ids, n, W, (size_t)-1, out, cap, out_bytes);
    return BFSC_REF_OK;
}

static int compress_rule(int codec, const void *ids, size_t n, int W, size_t thr,
                         uint8_t *out, size_t cap, size_t *out_bytes) {
    if ((W != 32 && W != 64) || !out || !out_bytes || (n && !ids)) return BFSC_REF_ERR_INVALID_ARG;
    if (codec != BFSC_REF_CODEC_PFOR && codec != BFSC_REF_CODEC_BP128) return BFSC_REF_ERR_INVALID_ARG;
    if (is_raw(n, W, thr)) {
        size_t body = n * (size_t)(W / 8), total = 32 + align_up(body, 16);
        if (total > cap) return BFSC_REF_ERR_DST_TOO_SMALL;
        write_header(out, W, 0, n, total, 0);
        memset(out + 32, 0, total - 32);
        for (size_t i = 0; i < n; i++) st_le(out + 32 + i * (W / 8), load_id(ids, i, W), W / 8);
        *out_bytes = total;
        return BFSC_REF_OK;
    }
    size_t nb = n_blocks(n);                                  /* O2 */
    size_t off = 32 + dir_bytes(nb);
    if (off > cap) return BFSC_REF_ERR_DST_TOO_SMALL;
    memset(out + 32, 0, dir_bytes(nb));
    uint8_t tmp[2304];
    for (size_t k = 0; k < nb; k++) {
        int m = (int)((n - BLK * k) < BLK ? (n - BLK * k) : BLK);
        uint64_t d[BLK];
        const uint8_t *xb = (const uint8_t *)ids + BLK * k * (size_t)(W / 8);
        uint64_t base = bfsc_ref_block_deltas(xb, m, W, d);   /* O3 */
        int n_exc = 0, b;
        if (codec == BFSC_REF_CODEC_BP128) b = bfsc_ref_choose_b_bp128(d);   /* FORMAT.md §7 */
        else b = bfsc_ref_choose_b(d, W, &n_exc);             /* O4, O5 */
        (void)n_exc;
        size_t sz = bfsc_ref_emit_block(d, base, b, W, tmp);  /* O6 */
        if (off + sz > cap) return BFSC_REF_ERR_DST_TOO_SMALL;
        memcpy(out + off, tmp, sz);
        st_le(out + 32 + 4 * k, off / 16, 4);                 /* O7: directory */
        off += sz;
    }
    st_le(out + 32 + 4 * nb, off / 16, 4);
    write_header(out, W, codec, n, off, (uint32_t)nb);     /* mode byte = codec (1 PFOR-D1, 2 BP128-D1) */
    *out_bytes = off;
    return BFSC_REF_OK;
}

/* Decode one block at `blk` with at most `avail` bytes; writes m IDs. */
static int decode_block(const uint8_t *blk, size_t avail, int W, int m, void *ids, size_t at) {
    if (avail < 16) return BFSC_REF_ERR_CORRUPT;
    uint64_t base = ld_le(blk, 8);
    int b = blk[8], n_exc = blk[9];
    if (b > W || n_exc > 127) return BFSC_REF_ERR_CORRUPT;
    if (bfsc_ref_block_bytes(b, n_exc, W) > avail) return BFSC_REF_ERR_CORRUPT;
    const uint8_t *payload = blk + 16;
    uint64_t d[BLK];
    for (int j = 0; j < BLK; j++) {
        int c = j % 4, r = j / 4;
        uint64_t v = 0;
        for (int i = 0; i < b; i++) {
            int s = r * b + i, word = s / 32, bit = s % 32;
            if ((payload[16 * word + 4 * c + bit / 8] >> (bit % 8)) & 1) v |= (uint64_t)1 << i;
        }
        d[j] = v;
    }
    if (n_exc > 0) {
        const uint8_t *e = payload + 16 * (size_t)b;
        const uint8_t *h = e + align_up((size_t)n_exc, (size_t)W / 8);
        for (int i = 0; i < n_exc; i++) {
            int p = e[i];
            if (p >= BLK) return BFSC_REF_ERR_CORRUPT;
            if (i > 0 && p <= e[i - 1]) return BFSC_REF_ERR_CORRUPT;   /* FORMAT.md §4: strictly ascending */
            uint64_t high = ld_le(h + (size_t)i * (W / 8), W / 8);
            if (b < 64) d[p] |= high << b;
        }
    }
    uint64_t mask = wmask(W), v = base & mask;
    for (int j = 0; j < m; j++) { v = (v + d[j]) & mask; store_id(ids, at + (size_t)j, W, v); }
    return BFSC_REF_OK;
}

/* Validates the stream header; returns mode/n/total/nb. */
static int parse_header(const uint8_t *in, size_t in_bytes, int W,
                        int *mode, uint64_t *n, uint64_t *total, uint64_t *nb) {
    if (in_bytes < 32) return BFSC_REF_ERR_CORRUPT;
    if (in[0] != 'B' || in[1] != 'F' || in[2] != 'S' || in[3] != 'C') return BFSC_REF_ERR_CORRUPT;
    if (in[4] != 1 || in[5] != W || in[6] > 2 || in[7] != 0) return BFSC_REF_ERR_CORRUPT;   /* FORMAT.md §4: reserved byte 7 */
    *mode = in[6];
    *n = ld_le(in + 8, 8); *total = ld_le(in + 16, 8); *nb = ld_le(in + 24, 4);
    if (*total > in_bytes || *total % 16 || *total < 32) return BFSC_REF_ERR_CORRUPT;
    if (*mode == 0) {
        if (*nb != 0) return BFSC_REF_ERR_CORRUPT;
        if (*n > (*total - 32) / (uint64_t)(W / 8)) return BFSC_REF_ERR_CORRUPT;
    } else {
        if (*nb != (*n + BLK - 1) / BLK) return BFSC_REF_ERR_CORRUPT;
        if (32 + dir_bytes(*nb) > *total) return BFSC_REF_ERR_CORRUPT;
    }
    return BFSC_REF_OK;
}

int bfsc_ref_decompress(const uint8_t *in, size_t in_bytes, int W,
                        void *ids, size_t ids_cap, size_t *n_ids) {
    if ((W != 32 && W != 64) || !in || !n_ids) return BFSC_REF_ERR_INVALID_ARG;
    int mode; uint64_t n, total, nb;
    int rc = parse_header(in, in_bytes, W, &mode, &n, &total, &nb);
    if (rc) return rc;
    if (n > ids_cap) return BFSC_REF_ERR_DST_TOO_SMALL;
    if (mode == 0) {
        for (size_t i = 0; i < n; i++) store_id(ids, i, W, ld_le(in + 32 + i * (W / 8), W / 8));
        *n_ids = n;
        return BFSC_REF_OK;
    }
    const uint8_t *dir = in + 32;
    uint64_t lo = (32 + dir_bytes(nb)) / 16;
    for (uint64_t k = 0; k < nb; k++) {
        uint64_t o0 = ld_le(dir + 4 * k, 4), o1 = ld_le(dir + 4 * (k + 1), 4);
        if (o0 < lo || o1 <= o0 || o1 > total / 16) return BFSC_REF_ERR_CORRUPT;
        int m = (int)((n - BLK * k) < BLK ? (n - BLK * k) : BLK);
        rc = decode_block(in + 16 * o0, 16 * (o1 - o0), W, m, ids, BLK * k);
        if (rc) return rc;
    }
    *n_ids = n;
    return BFSC_REF_OK;
}

int bfsc_ref_compress_batch(const void *ids, const uint64_t *in_off, size_t n_buf, int W,
                            size_t thr, uint8_t *out, size_t cap, uint64_t *out_off) {
    return bfsc_ref_compress_batch_codec(BFSC_REF_CODEC_PFOR, ids, in_off, n_buf, W, thr, out, cap, out_off);
}

int bfsc_ref_compress_batch_codec(int codec, const void *ids, const uint64_t *in_off, size_t n_buf, int W,
                                  size_t thr, uint8_t *out, size_t cap, uint64_t *out_off) {
    if (!in_off || !out_off) return BFSC_REF_ERR_INVALID_ARG;
    size_t off = 0;
    for (size_t i = 0; i < n_buf; i++) {
        size_t bytes = 0;
        const uint8_t *src = (const uint8_t *)ids + in_off[i] * (size_t)(W / 8);
        int rc = bfsc_ref_compress_codec(codec, src, in_off[i + 1] - in_off[i], W, thr, out + off, cap - off, &bytes);
        if (rc) return rc;
        out_off[i] = off;
        off += bytes;
    }
    out_off[n_buf] = off;
    return BFSC_REF_OK;
}

int bfsc_ref_decompress_batch(const uint8_t *in, const uint64_t *in_off, size_t n_buf, int W,
                              void *ids, size_t ids_cap, uint64_t *id_off) {
    if (!in_off || !id_off) return BFSC_REF_ERR_INVALID_ARG;
    size_t at = 0;
    for (size_t i = 0; i < n_buf; i++) {
        size_t n = 0;
        uint8_t *dst = (uint8_t *)ids + at * (size_t)(W / 8);
        int rc = bfsc_ref_decompress(in + in_off[i], in_off[i + 1] - in_off[i], W, dst, ids_cap - at, &n);
        if (rc) return rc;
        id_off[i] = at;
        at += n;
    }
    id_off[n_buf] = at;
    return BFSC_REF_OK;
}

/* ---- frontier bitmaps (FORMAT.md §9; "32-bit-word bitmap", Algorithm 4 line 11, L1381-1392, L2080) ----
 * A frontier given as a bitmap: bit v of the bitmap (bit v % 32 of 32-bit little-endian word v / 32) set <=> vertex
 * id_base + v is in the frontier. The stream of a bitmap is, by definition, the stream of its sorted ID list. */
int bfsc_ref_compress_bitmap(int codec, const uint32_t *bitmap, size_t n_bits, uint64_t id_base, int W, size_t thr,
                             uint8_t *out, size_t cap, size_t *out_bytes) {
    if ((W != 32 && W != 64) || (n_bits && !bitmap)) return BFSC_REF_ERR_INVALID_ARG;
    size_t n = 0;
    for (size_t v = 0; v < n_bits; v++) n += (bitmap[v / 32] >> (v % 32)) & 1u;
    void *ids = malloc((n ? n : 1) * (size_t)(W / 8));
    if (!ids) return BFSC_REF_ERR_INVALID_ARG;
    size_t k = 0;
    for (size_t v = 0; v < n_bits; v++)                        /* ascending bit index = ascending ID */
        if ((bitmap[v / 32] >> (v % 32)) & 1u) store_id(ids, k++, W, (id_base + v) & wmask(W));
    int rc = bfsc_ref_compress_codec(codec, ids, n, W, thr, out, cap, out_bytes);
    free(ids);
    return rc;
}

/* Decode, then OR bit (x - id_base) into the bitmap for every decoded ID x (the "t ⊙ ¬Π" consumer of Algorithm 4
 * works on bitmaps). An ID outside [id_base, id_base + n_bits) does not fit the bitmap: DST_TOO_SMALL. *n_ids = IDs decoded. */
int bfsc_ref_decompress_to_bitmap(const uint8_t *in, size_t in_bytes, int W, uint64_t id_base,
                                  uint32_t *bitmap, size_t n_bits, size_t *n_ids) {
    if ((W != 32 && W != 64) || !in || !n_ids) return BFSC_REF_ERR_INVALID_ARG;
    int mode; uint64_t n, total, nb;
    int rc = parse_header(in, in_bytes, W, &mode, &n, &total, &nb);
    if (rc) return rc;
    void *ids = malloc((n ? n : 1) * (size_t)(W / 8));
    if (!ids) return BFSC_REF_ERR_INVALID_ARG;
    size_t got = 0;
    rc = bfsc_ref_decompress(in, in_bytes, W, ids, n, &got);
    for (size_t i = 0; !rc && i < got; i++) {
        uint64_t v = (load_id(ids, i, W) - id_base) & wmask(W);
        if (v >= n_bits) rc = BFSC_REF_ERR_DST_TOO_SMALL;
    }
    for (size_t i = 0; !rc && i < got; i++) {
        uint64_t v = (load_id(ids, i, W) - id_base) & wmask(W);
        bitmap[v / 32] |= 1u << (v % 32);
    }
    free(ids);
    if (!rc) *n_ids = got;
    return rc;
}

/* FORMAT.md §10: a (visited) bitmap as a container that lists its MINORITY bits — the set bits if there are at most as
 * many of them as clear ones, else the clear bits — as one stream of §1 (u32 bit indices, threshold 0), or holds the
 * bitmap itself (kind 0) when the stream would not be smaller. PAPER.md L2065, L2104-2113, L2166: the zone the thesis
 * left uncompressed; the thesis gives no algorithm (reading 12). cap >= bfsc_ref_vbitmap_bound(n_bits). */
size_t bfsc_ref_vbitmap_bound(size_t n_bits) {
    size_t words = (n_bits + 31) / 32;
    return 32 + (4 * words + 15) / 16 * 16;
}

int bfsc_ref_compress_vbitmap(int codec, const uint32_t *bitmap, size_t n_bits, uint8_t *out, size_t cap, size_t *out_bytes) {
    if (!out || !out_bytes || (n_bits && !bitmap) || n_bits > ((size_t)1 << 32)) return BFSC_REF_ERR_INVALID_ARG;
    size_t words = (n_bits + 31) / 32, raw = (4 * words + 15) / 16 * 16;
    if (cap < 32 + raw) return BFSC_REF_ERR_DST_TOO_SMALL;
    size_t k = 0;
    for (size_t v = 0; v < n_bits; v++) k += (bitmap[v / 32] >> (v % 32)) & 1u;
    int list_set = k <= n_bits - k;                                  /* the minority; a tie lists the set bits */
    size_t n = list_set ? k : n_bits - k, j = 0;
    uint32_t *ids = malloc((n ? n : 1) * sizeof(uint32_t));
    size_t scap = bfsc_ref_compress_bound(n, 32);
    uint8_t *stream = malloc(scap);
    if (!ids || !stream) { free(ids); free(stream); return BFSC_REF_ERR_INVALID_ARG; }
    for (size_t v = 0; v < n_bits; v++)
        if ((int)((bitmap[v / 32] >> (v % 32)) & 1u) == list_set) ids[j++] = (uint32_t)v;
    size_t sb = 0;
    int rc = bfsc_ref_compress_codec(codec, ids, n, 32, 0, stream, scap, &sb);
    free(ids);
    if (rc) { free(stream); return rc; }
    int kind = sb < raw ? (list_set ? 1 : 2) : 0;                    /* not smaller than the bitmap itself: kind 0 */
    size_t payload = kind ? sb : raw;
    memset(out, 0, 32 + payload);
    out[0] = 'B'; out[1] = 'F'; out[2] = 'S'; out[3] = 'V';
    out[4] = 1; out[5] = 32; out[6] = (uint8_t)kind; out[7] = 0;
    st_le(out + 8, n_bits, 8);
    st_le(out + 16, 32 + payload, 8);
    st_le(out + 24, kind ? n : 0, 8);
    if (kind) memcpy(out + 32, stream, sb);
    else
        for (size_t v = 0; v < n_bits; v++)                          /* bits >= n_bits stay 0 */
            if ((bitmap[v / 32] >> (v % 32)) & 1u) out[32 + v / 8] |= (uint8_t)(1u << (v % 8));
    free(stream);
    *out_bytes = 32 + payload;
    return BFSC_REF_OK;
}

/* The bitmap is overwritten (every word up to ceil(n_bits / 32); bits >= n_bits are 0). Nothing is changed on an error. */
int bfsc_ref_decompress_vbitmap(const uint8_t *in, size_t in_bytes, uint32_t *bitmap, size_t n_bits) {
    if (!in || (n_bits && !bitmap)) return BFSC_REF_ERR_INVALID_ARG;
    if (in_bytes < 32) return BFSC_REF_ERR_CORRUPT;
    if (in[0] != 'B' || in[1] != 'F' || in[2] != 'S' || in[3] != 'V') return BFSC_REF_ERR_CORRUPT;
    if (in[4] != 1 || in[5] != 32 || in[6] > 2 || in[7] != 0) return BFSC_REF_ERR_CORRUPT;
    uint64_t nbits = ld_le(in + 8, 8), total = ld_le(in + 16, 8), n_listed = ld_le(in + 24, 8);
    int kind = in[6];
    if (total > in_bytes || total % 16 || total < 32) return BFSC_REF_ERR_CORRUPT;
    if (nbits != n_bits) return BFSC_REF_ERR_DST_TOO_SMALL;
    size_t words = (n_bits + 31) / 32, raw = (4 * words + 15) / 16 * 16;
    uint32_t *res = calloc(words ? words : 1, sizeof(uint32_t));
    if (!res) return BFSC_REF_ERR_INVALID_ARG;
    int rc = BFSC_REF_OK;
    if (kind == 0) {
        if (total != 32 + raw || n_listed != 0) rc = BFSC_REF_ERR_CORRUPT;
        for (size_t v = 0; !rc && v < 8 * raw; v++) {
            unsigned bit = (in[32 + v / 8] >> (v % 8)) & 1u;
            if (v >= n_bits) { if (bit) rc = BFSC_REF_ERR_CORRUPT; }     /* the pad is zero */
            else if (bit) res[v / 32] |= 1u << (v % 32);
        }
    } else {
        size_t got = 0;
        rc = bfsc_ref_decompress_to_bitmap(in + 32, (size_t)total - 32, 32, 0, res, n_bits, &got);
        if (rc == BFSC_REF_ERR_DST_TOO_SMALL) rc = BFSC_REF_ERR_CORRUPT;   /* an ID >= n_bits inside the container */
        if (!rc && got != n_listed) rc = BFSC_REF_ERR_CORRUPT;
        if (!rc && kind == 2)
            for (size_t v = 0; v < n_bits; v++) res[v / 32] ^= 1u << (v % 32);
    }
    if (!rc) memcpy(bitmap, res, words * sizeof(uint32_t));
    free(res);
    return rc;
}

/* Algorithm 4, lines 10-13, with the frontier t and the visited set of Pi as bitmaps:
 *   line 10  t <- decompress(t'')          the decoded IDs
 *   line 11  t <- t (.) not Pi             keep those not visited yet
 *   line 12  Pi <- Pi + t                  mark them visited
 *   line 13  f <- t                        they are (part of) the next frontier: OR-ed into `frontier`
 * One ID at a time, in stream order; an ID met a second time is visited by then and changes nothing. */
int bfsc_ref_decompress_to_frontier(const uint8_t *in, size_t in_bytes, int W, uint64_t id_base,
                                    uint32_t *frontier, uint32_t *visited, size_t n_bits, size_t *n_ids) {
    if ((W != 32 && W != 64) || !in || !n_ids || !frontier || !visited) return BFSC_REF_ERR_INVALID_ARG;
    int mode; uint64_t n, total, nb;
    int rc = parse_header(in, in_bytes, W, &mode, &n, &total, &nb);
    if (rc) return rc;
    void *ids = malloc((n ? n : 1) * (size_t)(W / 8));
    if (!ids) return BFSC_REF_ERR_INVALID_ARG;
    size_t got = 0;
    rc = bfsc_ref_decompress(in, in_bytes, W, ids, n, &got);
    for (size_t i = 0; !rc && i < got; i++) {
        uint64_t v = (load_id(ids, i, W) - id_base) & wmask(W);
        if (v >= n_bits) rc = BFSC_REF_ERR_DST_TOO_SMALL;
    }
    for (size_t i = 0; !rc && i < got; i++) {
        uint64_t v = (load_id(ids, i, W) - id_base) & wmask(W);
        uint32_t bit = 1u << (v % 32);
        if (!(visited[v / 32] & bit)) {                          /* line 11 */
            visited[v / 32] |= bit;                              /* line 12 */
            frontier[v / 32] |= bit;                             /* line 13 */
        }
    }
    free(ids);
    if (!rc) *n_ids = got;
    return rc;
}

/* ------------------------------------------------------------------------------------
 * Multi-threaded drivers (bench.py cpu_baseline only). Work unit = one 128-ID block, run
 * through the very same scalar routines; three phases: block sizes -> serial prefix ->
 * emit. Output bytes are identical to the serial functions.
 * ---------------------------------------------------------------------------------- */
typedef struct {
    /* shared */
    const void *ids; const uint64_t *in_off; size_t n_buf; int W; size_t thr;
    uint8_t *out; uint64_t *out_off;
    const uint64_t *blk_first;   /* n_buf+1: first global block index of each buffer (0 blocks if raw) */
    uint32_t *blk_size;          /* per global block: bytes */
    uint8_t *blk_b;              /* per global block: chosen b */
    uint64_t *blk_off;           /* per global block: absolute byte offset in out */
    const uint8_t *in; void *ids_out; const uint64_t *id_off;   /* decode */
    int phase, rc;
    size_t lo, hi;               /* this thread's range (blocks or buffers) */
} mt_job;

static size_t find_buf(const uint64_t *blk_first, size_t n_buf, uint64_t g) {
    size_t lo = 0, hi = n_buf;           /* largest i with blk_first[i] <= g and blk_first[i+1] > g */
    while (hi - lo > 1) { size_t mid = (lo + hi) / 2; if (blk_first[mid] <= g) lo = mid; else hi = mid; }
    while (blk_first[lo + 1] <= g) lo++;
    return lo;
}

static void *mt_worker(void *arg) {
    mt_job *j = (mt_job *)arg;
    int W = j->W; size_t eb = (size_t)(W / 8);
    if (j->phase == 0 || j->phase == 2) {                   /* per block: size / emit */
        for (size_t g = j->lo; g < j->hi; g++) {
            size_t i = find_buf(j->blk_first, j->n_buf, g);
            size_t k = g - j->blk_first[i], n = j->in_off[i + 1] - j->in_off[i];
            int m = (int)((n - BLK * k) < BLK ? (n - BLK * k) : BLK);
            const uint8_t *xb = (const uint8_t *)j->ids + (j->in_off[i] + BLK * k) * eb;
            uint64_t d[BLK];
            uint64_t base = bfsc_ref_block_deltas(xb, m, W, d);
            if (j->phase == 0) {
                int n_exc, b = bfsc_ref_choose_b(d, W, &n_exc);
                j->blk_b[g] = (uint8_t)b;
                j->blk_size[g] = (uint32_t)bfsc_ref_block_bytes(b, n_exc, W);
            } else {
                bfsc_ref_emit_block(d, base, j->blk_b[g], W, j->out + j->blk_off[g]);
            }
        }
    } else if (j->phase == 3) {                             /* per buffer: header, directory, raw */
        for (size_t i = j->lo; i < j->hi; i++) {
            size_t n = j->in_off[i + 1] - j->in_off[i];
            uint8_t *s = j->out + j->out_off[i];
            size_t total = j->out_off[i + 1] - j->out_off[i];
            if (is_raw(n, W, j->thr)) {
                size_t bytes = 0;
                int rc = bfsc_ref_compress((const uint8_t *)j->ids + j->in_off[i] * eb, n, W, j->thr, s, total, &bytes);
                if (rc) j->rc = rc;
                continue;
            }
            size_t nb = n_blocks(n);
            memset(s + 32, 0, dir_bytes(nb));
            for (size_t k = 0; k < nb; k++) st_le(s + 32 + 4 * k, (j->blk_off[j->blk_first[i] + k] - j->out_off[i]) / 16, 4);
            st_le(s + 32 + 4 * nb, total / 16, 4);
            write_header(s, W, 1, n, total, (uint32_t)nb);
        }
    } else if (j->phase == 4) {                             /* decode, per buffer */
        for (size_t i = j->lo; i < j->hi; i++) {
            size_t n = 0;
            int rc = bfsc_ref_decompress(j->in + j->in_off[i], j->in_off[i + 1] - j->in_off[i], W,
                                         (uint8_t *)j->ids_out + j->id_off[i] * eb,
                                         j->id_off[i + 1] - j->id_off[i], &n);
            if (rc) j->rc = rc;
        }
    } else if (j->phase == 5) {                             /* decode, per block of ONE stream */
        const uint8_t *in = j->in; const uint8_t *dir = in + 32;
        uint64_t n = ld_le(in + 8, 8), total = ld_le(in + 16, 8), nb = ld_le(in + 24, 4);
        uint64_t lo16 = (32 + dir_bytes(nb)) / 16;
        for (size_t k = j->lo; k < j->hi; k++) {
            uint64_t o0 = ld_le(dir + 4 * k, 4), o1 = ld_le(dir + 4 * (k + 1), 4);
            if (o0 < lo16 || o1 <= o0 || o1 > total / 16) { j->rc = BFSC_REF_ERR_CORRUPT; return 0; }
            int m = (int)((n - BLK * k) < BLK ? (n - BLK * k) : BLK);
            int rc = decode_block(in + 16 * o0, 16 * (o1 - o0), W, m, j->ids_out, BLK * k);
            if (rc) { j->rc = rc; return 0; }
        }
    }
    return 0;
}

static int run_phase(mt_job *tmpl, int phase, size_t total, int threads) {
    if (threads < 1) threads = 1;
    if ((size_t)threads > total) threads = total ? (int)total : 1;
    pthread_t *th = (pthread_t *)malloc(sizeof(pthread_t) * (size_t)threads);
    mt_job *jobs = (mt_job *)malloc(sizeof(mt_job) * (size_t)threads);
    for (int t = 0; t < threads; t++) {
        jobs[t] = *tmpl; jobs[t].phase = phase; jobs[t].rc = 0;
        jobs[t].lo = total * (size_t)t / (size_t)threads;
        jobs[t].hi = total * (size_t)(t + 1) / (size_t)threads;
        if (threads == 1) mt_worker(&jobs[t]); else pthread_create(&th[t], 0, mt_worker, &jobs[t]);
    }
    int rc = 0;
    for (int t = 0; t < threads; t++) {
        if (threads > 1) pthread_join(th[t], 0);
        if (jobs[t].rc) rc = jobs[t].rc;
    }
    free(th); free(jobs);
    return rc;
}

int bfsc_ref_compress_batch_mt(const void *ids, const uint64_t *in_off, size_t n_buf, int W,
                               size_t thr, uint8_t *out, size_t cap, uint64_t *out_off, int threads) {
    if (!in_off || !out_off || (W != 32 && W != 64)) return BFSC_REF_ERR_INVALID_ARG;
    uint64_t *blk_first = (uint64_t *)malloc(sizeof(uint64_t) * (n_buf + 1));
    uint64_t g = 0;
    for (size_t i = 0; i < n_buf; i++) {
        size_t n = in_off[i + 1] - in_off[i];
        blk_first[i] = g;
        if (!is_raw(n, W, thr)) g += n_blocks(n);
    }
    blk_first[n_buf] = g;
    uint32_t *blk_size = (uint32_t *)malloc(sizeof(uint32_t) * (g + 1));
    uint8_t *blk_b = (uint8_t *)malloc(g + 1);
    uint64_t *blk_off = (uint64_t *)malloc(sizeof(uint64_t) * (g + 1));
    mt_job t; memset(&t, 0, sizeof t);
    t.ids = ids; t.in_off = in_off; t.n_buf = n_buf; t.W = W; t.thr = thr; t.out = out; t.out_off = out_off;
    t.blk_first = blk_first; t.blk_size = blk_size; t.blk_b = blk_b; t.blk_off = blk_off;
    int rc = run_phase(&t, 0, g, threads);
    size_t off = 0;                                          /* serial prefix */
    for (size_t i = 0; i < n_buf && !rc; i++) {
        size_t n = in_off[i + 1] - in_off[i];
        out_off[i] = off;
        if (is_raw(n, W, thr)) { off += 32 + align_up(n * (size_t)(W / 8), 16); }
        else {
            off += 32 + dir_bytes(n_blocks(n));
            for (uint64_t q = blk_first[i]; q < blk_first[i + 1]; q++) { blk_off[q] = off; off += blk_size[q]; }
        }
        if (off > cap) rc = BFSC_REF_ERR_DST_TOO_SMALL;
    }
    out_off[n_buf] = off;
    if (!rc) rc = run_phase(&t, 2, g, threads);
    if (!rc) rc = run_phase(&t, 3, n_buf, threads);
    free(blk_first); free(blk_size); free(blk_b); free(blk_off);
    return rc;
}

int bfsc_ref_decompress_batch_mt(const uint8_t *in, const uint64_t *in_off, size_t n_buf, int W,
                                 void *ids, size_t ids_cap, uint64_t *id_off, int threads) {
    if (!in_off || !id_off || (W != 32 && W != 64)) return BFSC_REF_ERR_INVALID_ARG;
    size_t at = 0;                                           /* serial: read n from each header */
    for (size_t i = 0; i < n_buf; i++) {
        int mode; uint64_t n, total, nb;
        int rc = parse_header(in + in_off[i], in_off[i + 1] - in_off[i], W, &mode, &n, &total, &nb);
        if (rc) return rc;
        id_off[i] = at; at += n;
    }
    id_off[n_buf] = at;
    if (at > ids_cap) return BFSC_REF_ERR_DST_TOO_SMALL;
    mt_job t; memset(&t, 0, sizeof t);
    t.in = in; t.in_off = in_off; t.n_buf = n_buf; t.W = W; t.ids_out = ids; t.id_off = id_off;
    if (n_buf == 1 && in[in_off[0] + 6] == 1) {              /* one big stream: split by blocks */
        t.in = in + in_off[0];
        return run_phase(&t, 5, ld_le(t.in + 24, 4), threads);
    }
    return run_phase(&t, 4, n_buf, threads);
}
