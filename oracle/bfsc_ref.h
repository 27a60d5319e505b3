/*
 * bfsc_ref — the ORACLE: a plain, scalar, obviously-correct CPU encoder/decoder for
 * the BFSC stream format (FORMAT.md v1).
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT. Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may call it. It shares no code,
 * header, table or helper with the CUDA path (paper_1704_00513_b200/csrc/), and the
 * CUDA path never calls it.
 *
 * What it computes, following /root/reference/PAPER.md (arxiv 1704.00513):
 *   - delta ("d-gap") coding of a sorted ID sequence ............ §5.1
 *   - frame-of-reference width ceil(log2(max+1-min)) ............ eq. (6)
 *   - binary packing in blocks of 128 with per-block width b .... L987-998, L1052-1056
 *   - patched coding: values >= 2^b are stored apart ............ eq. (8)/(9), L1000-1011
 *   - compression threshold (minimum size that triggers it) ..... §5.4.3
 * The byte layout is FORMAT.md's (the paper gives none); each ◆ reading is listed in
 * DESIGN.md. The result is an encoding, so encode follows the algorithm step by step
 * (SURVEY.md §8(c) O1-O7); decode is the plain definition of the format's semantics.
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): the paper's worked widths (eq. 7, eq. 9),
 * closed-form sizes for constant-gap sequences, brute-force choice of b written
 * independently in Python, an independent pure-Python big-integer decoder
 * (oracle/witness.py) built from FORMAT.md alone, hand-computed byte vectors,
 * round-trip identity and the walk-the-headers invariants. Mode 2 (BP128-D1, FORMAT.md §7): hand-evaluated
 * sizes (tests/golden/bp128_sizes.txt), b = int.bit_length of the widest delta, blocks byte-equal to the
 * witness builder with that b, witness decode, equality with mode 1 where no exception pays.
 * Parity vs the thesis's own codec (S4-BP128 bytes / ratios): parity unpinned — the
 * thesis ships no byte layout and its sample data are not available.
 *
 * All arithmetic is integer (u32/u64, modular). W is 32 or 64.
 */
#ifndef BFSC_REF_H
#define BFSC_REF_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

enum {
    BFSC_REF_OK = 0,
    BFSC_REF_ERR_INVALID_ARG = 1,
    BFSC_REF_ERR_DST_TOO_SMALL = 2,
    BFSC_REF_ERR_CORRUPT = 3
};

/* Encoder rule = mode byte of the stream it writes (FORMAT.md §1, §7). BFSC_REF_FLAG_RAW_FALLBACK, OR-ed into
 * the rule: a stream that the rule does not make smaller than its RAW form is sent RAW (FORMAT.md §8). */
enum { BFSC_REF_CODEC_PFOR = 1, BFSC_REF_CODEC_BP128 = 2, BFSC_REF_FLAG_RAW_FALLBACK = 0x200 };

/* bit length of v: 0 for 0, floor(log2 v)+1 otherwise. For a range [min,max] the FOR
 * width of eq. (6) is bfsc_ref_width(max - min). */
int bfsc_ref_width(uint64_t v);

/* FORMAT.md §2: 16 + 16 b + (n_exc ? align16(align_{W/8}(n_exc) + n_exc W/8) : 0) */
size_t bfsc_ref_block_bytes(int b, int n_exc, int W);

/* FORMAT.md §3 */
size_t bfsc_ref_compress_bound(size_t n, int W);

/* Deltas of one block (FORMAT.md §2 "Deltas"): x points at the block's first ID, m valid
 * IDs (1..128); d[128] is written (d[0]=0, zero padded). Returns base = x[0]. */
uint64_t bfsc_ref_block_deltas(const void *x, int m, int W, uint64_t d[128]);

/* Canonical b for 128 deltas (FORMAT.md §2 "Choice of b"): argmin of block_bytes over
 * b in 0..maxw, ties to the largest b. Writes n_exc(b). */
int bfsc_ref_choose_b(const uint64_t d[128], int W, int *n_exc);

/* b of the no-exception codec (FORMAT.md §7, mode 2 = BP128-D1; the thesis's codec class S4-BP128,
 * PAPER.md L1052-1056): the width of the block's widest delta; n_exc = 0. */
int bfsc_ref_choose_b_bp128(const uint64_t d[128]);

/* Emit one block with a GIVEN b (any 0..W): header, payload, exceptions, pads.
 * Returns its byte count (= block_bytes(b, n_exc(b))). out must hold 16+16W+... bytes
 * (<= 16 + 16*64 + 16 + 127*9 rounded; 2304 is always enough). */
size_t bfsc_ref_emit_block(const uint64_t d[128], uint64_t base, int b, int W, uint8_t *out);

/* One stream. Returns BFSC_REF_OK and *out_bytes, or an error. */
int bfsc_ref_compress(const void *ids, size_t n, int W, size_t raw_threshold_bytes,
                      uint8_t *out, size_t out_capacity, size_t *out_bytes);

/* Same, with the encoder rule given: BFSC_REF_CODEC_PFOR (what bfsc_ref_compress does) or
 * BFSC_REF_CODEC_BP128 (every block b = maxw, no exceptions; header mode 2). */
int bfsc_ref_compress_codec(int codec, const void *ids, size_t n, int W, size_t raw_threshold_bytes,
                            uint8_t *out, size_t out_capacity, size_t *out_bytes);
int bfsc_ref_compress_batch_codec(int codec, const void *ids, const uint64_t *in_offsets, size_t n_buf, int W,
                                  size_t raw_threshold_bytes,
                                  uint8_t *out, size_t out_capacity, uint64_t *out_offsets);

/* One stream. in_bytes = bytes available at `in` (may exceed the stream's total_bytes).
 * Writes *n_ids; ids must hold ids_capacity elements of W bits. */
int bfsc_ref_decompress(const uint8_t *in, size_t in_bytes, int W,
                        void *ids, size_t ids_capacity, size_t *n_ids);

/* Batches (FORMAT.md §5). in_offsets: n_buf+1 element offsets into ids.
 * out_offsets: n_buf+1 byte offsets, written. */
int bfsc_ref_compress_batch(const void *ids, const uint64_t *in_offsets, size_t n_buf, int W,
                            size_t raw_threshold_bytes,
                            uint8_t *out, size_t out_capacity, uint64_t *out_offsets);

/* in_offsets: n_buf+1 byte offsets into `in`; id_offsets: n_buf+1 element offsets, written. */
int bfsc_ref_decompress_batch(const uint8_t *in, const uint64_t *in_offsets, size_t n_buf, int W,
                              void *ids, size_t ids_capacity, uint64_t *id_offsets);

/* Frontier bitmaps (FORMAT.md §9): bit v (bit v % 32 of word v / 32) <=> ID id_base + v. compress_bitmap = compress
 * of the ascending ID list of the set bits; decompress_to_bitmap ORs the decoded IDs' bits into the bitmap
 * (DST_TOO_SMALL if an ID lies outside [id_base, id_base + n_bits)). */
int bfsc_ref_compress_bitmap(int codec, const uint32_t *bitmap, size_t n_bits, uint64_t id_base, int W,
                             size_t raw_threshold_bytes, uint8_t *out, size_t out_capacity, size_t *out_bytes);
int bfsc_ref_decompress_to_bitmap(const uint8_t *in, size_t in_bytes, int W, uint64_t id_base,
                                  uint32_t *bitmap, size_t n_bits, size_t *n_ids);
/* FORMAT.md §10: a bitmap as a container that lists its minority bits (set or
 * clear) as one u32 stream, or holds the bitmap itself when that is not smaller. cap >= bfsc_ref_vbitmap_bound(n_bits). */
size_t bfsc_ref_vbitmap_bound(size_t n_bits);
int bfsc_ref_compress_vbitmap(int codec, const uint32_t *bitmap, size_t n_bits, uint8_t *out, size_t out_capacity,
                              size_t *out_bytes);
int bfsc_ref_decompress_vbitmap(const uint8_t *in, size_t in_bytes, uint32_t *bitmap, size_t n_bits);
/* Algorithm 4 lines 10-13 on bitmaps: for the decoded IDs S,
 * frontier |= S \ visited and visited |= S (FORMAT.md §9, last item). Nothing is changed on an error. */
int bfsc_ref_decompress_to_frontier(const uint8_t *in, size_t in_bytes, int W, uint64_t id_base,
                                    uint32_t *frontier, uint32_t *visited, size_t n_bits, size_t *n_ids);

/* Multi-threaded drivers used only by bench.py's cpu_baseline leg: independent buffers
 * are spread over `threads` pthreads; each buffer goes through the same scalar routines
 * above. A single large stream is split into contiguous runs of blocks
 * (sizes -> prefix -> pack), every run through the same scalar block routines.
 * Byte-identical to the single-threaded functions. */
int bfsc_ref_compress_batch_mt(const void *ids, const uint64_t *in_offsets, size_t n_buf, int W,
                               size_t raw_threshold_bytes, uint8_t *out, size_t out_capacity,
                               uint64_t *out_offsets, int threads);
int bfsc_ref_decompress_batch_mt(const uint8_t *in, const uint64_t *in_offsets, size_t n_buf, int W,
                                 void *ids, size_t ids_capacity, uint64_t *id_offsets, int threads);

#ifdef __cplusplus
}
#endif
#endif
