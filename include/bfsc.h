/*
 * bfsc.h — C ABI of the B200 (sm_100a) BFS-frontier codec. The boundary of the product.
 *
 * Operation (arxiv 1704.00513 = /root/reference/PAPER.md): compress / decompress the BFS
 * frontier traffic — sorted vertex-ID queues (§4.1.4) — before / after each of
 * the two exchanges of a BFS level (Algorithm 4 lines 5-7 and 9-11, L1344-1379; call shape
 * compress(buffer)->bytes, decompress(bytes)->buffer of Algorithm 5), with
 * delta coding (L979-986) + frame-of-reference binary packing in blocks of 128 IDs with a
 * per-block width b (eq. 6) + patched exceptions (L1000-1011),
 * and a compression threshold below which a buffer is sent raw (§5.4.3).
 * The byte layout is FORMAT.md (version 1). The batch calls take the (buffer, counts/displs)
 * shape of the MPI ...V collectives the streams are sent with (L750-754); the size metadata
 * (out_offsets) is handed back to the caller, who exchanges it first (L1790).
 *
 * Conventions
 *  - Pointers named d_* are DEVICE pointers owned by the caller; h_* are HOST pointers.
 *    The library allocates nothing, frees nothing and never synchronises (except the *_host
 *    convenience calls, which synchronise `cuda_stream` before returning).
 *  - Every call enqueues its kernels on `cuda_stream` (a cudaStream_t passed as void*;
 *    NULL = the legacy default stream) and returns immediately. Stream order holds for
 *    everything a call reads or writes. The kernels are launched with programmatic dependent
 *    launch: a kernel may become resident while its predecessor in the stream still runs, but
 *    waits for that predecessor to complete before it touches memory (back-to-back calls pay
 *    no launch gap). Because a call only enqueues kernels, a sequence of calls may be captured
 *    in a CUDA graph (stream capture) and replayed, after one call of each kind outside the
 *    capture (one-time function attributes); the launch counter then counts the capture only.
 *  - Concurrency: calls may be issued from several host threads and on any streams of a device, also
 *    at the same time, each with a workspace of its own. The compress kernels run a device-wide scan of
 *    block sizes in which CTAs wait for one another; every tile of work is handed out by an atomic ticket,
 *    in order, so whatever a CTA waits for is held by a CTA that is already running: no kernel of this
 *    library assumes that its whole grid is resident (two compress grids, or a compress grid next to a
 *    foreign persistent kernel, cannot deadlock). Opt-out: BFSC_CODEC_FLAG_EXCLUSIVE (see bfsc_codec).
 *  - d_ids / d_out / d_in must be 16-byte aligned; element offsets inside a batch may be
 *    arbitrary (buffers that start off a 16-byte boundary are staged / written through
 *    aligned 16-byte chunks all the same). Nothing is read beyond the last ID of a buffer
 *    (its last, ragged 16-byte chunk is fetched partially) and nothing before d_ids.
 *  - IDs are little-endian unsigned integers of W = 32 or 64 bits (bfsc_dtype).
 *  - Return value: host-detectable errors only (null / misaligned pointer, bad dtype,
 *    workspace too small, launch failure -> BFSC_ERR_CUDA).
 *  - Data-dependent errors are written to *d_status (a device uint32, 0 = OK, first error
 *    wins; the caller zero-initialises it or passes the same word through a sequence of
 *    calls): BFSC_ERR_DST_TOO_SMALL (output / ids capacity exceeded: nothing is written
 *    beyond capacity), BFSC_ERR_CORRUPT (decoder: anything FORMAT.md §4 rejects),
 *    BFSC_ERR_INVALID_ARG (workspace too small for the block count found on the device,
 *    non-monotone offsets). On error the output content is unspecified, but no out-of-bounds
 *    access occurs. d_status may be NULL (errors are then dropped).
 *  - raw_threshold_bytes: a buffer is sent RAW iff n*W/8 < raw_threshold_bytes
 *    (FORMAT.md §1); 0 = always compress.
 *  - Workspace: bfsc_workspace_bytes(n_ids_total, n_buf, t) bytes (about 33 bytes per 128 IDs
 *    + 24 per buffer: scan states and, for batch calls, a table of where every block lives),
 *    16-byte aligned, any content on entry, clobbered by the call; one workspace per in-flight
 *    call (calls on the same stream may share one).
 *  - Compressed output is canonical: byte-identical to the scalar oracle (oracle/), pads
 *    included. The decoder accepts any well-formed stream.
 */
#ifndef BFSC_H
#define BFSC_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    BFSC_OK = 0,
    BFSC_ERR_INVALID_ARG = 1,
    BFSC_ERR_DST_TOO_SMALL = 2,
    BFSC_ERR_CORRUPT = 3,
    BFSC_ERR_CUDA = 4,
    BFSC_ERR_UNSUPPORTED = 5
} bfsc_status;

typedef enum { BFSC_U32 = 32, BFSC_U64 = 64 } bfsc_dtype;

/* Encoder rule of a compress call = mode byte of the streams it writes (FORMAT.md §1, §7):
 *   BFSC_CODEC_PFOR  (1) patched frame of reference: per block the b that minimises the block size,
 *                        values >= 2^b stored apart as exceptions — what
 *                        bfsc_compress / bfsc_compress_batch do;
 *   BFSC_CODEC_BP128 (2) plain binary packing, the codec class the thesis ran (S4-BP128, L1052-1056):
 *                        b = width of the block's widest delta (eq. 6), no exceptions. Skips
 *                        step E2's size argmin; one outlier widens its whole block (L1000).
 * Buffers below the raw threshold are RAW (mode 0) under either rule. bfsc_decompress[_batch] read
 * the mode from each stream header and decode every mode.
 *
 * Launch flag, OR-ed into the codec argument of the *_codec calls:
 *   BFSC_CODEC_FLAG_EXCLUSIVE  the caller vouches that nothing else occupies the device while the call runs
 *                        (no kernel on another stream, no second compress call in flight), so that the
 *                        whole compress grid becomes resident at once. The first two tiles of every CTA are
 *                        then assigned statically and start before the call's plan kernel has finished
 *                        (about 2 us less per call). If the promise is broken the call can deadlock.
 *                        The first tiles' IDs are also read BEFORE the call waits for the kernel enqueued before it
 *                        on the stream: d_ids must not be the output of the bfsc call enqueued immediately before
 *                        this one (bfsc kernels release their successor early; after any other kernel, an event
 *                        or a synchronisation the IDs are complete). Output bytes are the same with or without
 *                        the flag.
 *   BFSC_CODEC_FLAG_RAW_FALLBACK  FORMAT.md §8: a stream that the rule does not make smaller than
 *                        its RAW form is sent RAW (mode 0) after all: total_bytes <= 32 + align16(n W / 8) always.
 *                        Single-buffer calls (bfsc_compress_codec, bfsc_compress_bitmap); the batch calls return
 *                        BFSC_ERR_UNSUPPORTED (streams of a batch lie back to back: a stream that shrinks after the
 *                        fact would move every stream behind it). The input is read a second time only for the
 *                        streams that fall back. */
typedef enum { BFSC_CODEC_PFOR = 1, BFSC_CODEC_BP128 = 2, BFSC_CODEC_FLAG_EXCLUSIVE = 0x100,
               BFSC_CODEC_FLAG_RAW_FALLBACK = 0x200 } bfsc_codec;

/* library / format version: (format_version << 16) | abi_revision */
uint32_t bfsc_version(void);

/* Worst-case bytes of ONE stream of n_ids IDs, RAW or compressed (FORMAT.md §3). Host. */
size_t bfsc_compress_bound(size_t n_ids, bfsc_dtype t);

/* Sum of bfsc_compress_bound over a batch; h_counts = n_buf HOST element counts. */
size_t bfsc_batch_compress_bound(const uint64_t* h_counts, size_t n_buf, bfsc_dtype t);

/* Workspace bytes sufficient for any of the four device calls on a batch of n_buf buffers
 * holding n_ids_total IDs in total (single-buffer calls: n_buf = 1). Host. The batch calls size their launches by the
 * workspace they are given: a small batch (a BFS level of up to ~1 MB) with a workspace sized for ITS total runs in one
 * launch; the same batch with a workspace sized for the largest level of the run takes the general three-launch path. */
size_t bfsc_workspace_bytes(size_t n_ids_total, size_t n_buf, bfsc_dtype t);

/* ONE buffer: d_ids[0..n_ids) -> one stream at d_out; *d_out_bytes (device) = its
 * total_bytes. Steps E0-E5 of SURVEY.md §8(a): compress() of Algorithm 4 lines 5 / 9 and Algorithm 5
 * — D1 deltas (L979-986), per-block width (eq. 6),
 * exceptions (L1000-1011), RAW below the threshold (L1309-1334); layout FORMAT.md §1-§3. */
bfsc_status bfsc_compress(const void* d_ids, size_t n_ids, bfsc_dtype t, size_t raw_threshold_bytes,
                          void* d_out, size_t out_capacity, uint64_t* d_out_bytes,
                          void* d_workspace, size_t workspace_bytes, uint32_t* d_status,
                          void* cuda_stream);

/* bfsc_compress for callers that cannot allocate (code under CUDA graph capture, tight serving loops, harnesses that
 * forbid cudaMalloc): the same kernels, with the workspace in a device array that is part of the library image
 * (a file-scope `static __device__` array of BFSC_NOALLOC_SCRATCH_BYTES bytes: every GPU that loads the library holds it
 * until the process exits). The call allocates nothing, on the host or on the device.
 *   n_ids <= BFSC_NOALLOC_MAX_IDS, else BFSC_ERR_INVALID_ARG (nothing is enqueued); everything else as bfsc_compress,
 *   output bytes included.
 *   ALL no-alloc calls of a device share that one array: two of them that overlap on the GPU (two streams, or two host
 *   threads on two streams) race on it and produce garbage — issue them on one stream at a time. The array keeps the
 *   last call's contents; whatever must start at zero (tile states, ticket counter) is reset by the call's own plan
 *   kernel, as for a caller-owned workspace. */
#define BFSC_NOALLOC_MAX_IDS ((size_t)1 << 22)
#define BFSC_NOALLOC_SCRATCH_BYTES ((size_t)1088 * 1024)
bfsc_status bfsc_compress_noalloc(const void* d_ids, size_t n_ids, bfsc_dtype t, size_t raw_threshold_bytes,
                                  void* d_out, size_t out_capacity, uint64_t* d_out_bytes, uint32_t* d_status,
                                  void* cuda_stream);

/* bfsc_compress with the encoder rule given (any other value: BFSC_ERR_INVALID_ARG). */
bfsc_status bfsc_compress_codec(bfsc_codec codec, const void* d_ids, size_t n_ids, bfsc_dtype t,
                                size_t raw_threshold_bytes, void* d_out, size_t out_capacity,
                                uint64_t* d_out_bytes, void* d_workspace, size_t workspace_bytes,
                                uint32_t* d_status, void* cuda_stream);

/* ONE stream at d_in (in_bytes available, >= its total_bytes) -> d_ids[0..n); *d_n_ids
 * (device) = n. Steps D0-D5: decompress() of Algorithm 4 lines 7 / 11: unpack
 * (L987-998), patch the exceptions (L1011), prefix-sum the deltas (L979-986); FORMAT.md §4. */
bfsc_status bfsc_decompress(const void* d_in, size_t in_bytes, bfsc_dtype t,
                            void* d_ids, size_t ids_capacity, uint64_t* d_n_ids,
                            void* d_workspace, size_t workspace_bytes, uint32_t* d_status,
                            void* cuda_stream);

/* n_buf buffers in one launch sequence — the send buffers of one exchange (ALLGATHERV / ALLTOALLV counts and
 * displacements; "data transfer grouping", L1786-1800). d_in_offsets: n_buf+1
 * non-decreasing ELEMENT offsets into d_ids (device). Streams are written back to back at d_out (FORMAT.md §5);
 * d_out_offsets[0..n_buf] (device, written) are their BYTE offsets, [n_buf] = total: the size metadata
 * the caller exchanges first (L1790). */
bfsc_status bfsc_compress_batch(const void* d_ids, const uint64_t* d_in_offsets, size_t n_buf,
                                bfsc_dtype t, size_t raw_threshold_bytes,
                                void* d_out, size_t out_capacity, uint64_t* d_out_offsets,
                                void* d_workspace, size_t workspace_bytes, uint32_t* d_status,
                                void* cuda_stream);

/* bfsc_compress_batch with the encoder rule given (one rule for all buffers of the batch). */
bfsc_status bfsc_compress_batch_codec(bfsc_codec codec, const void* d_ids, const uint64_t* d_in_offsets,
                                      size_t n_buf, bfsc_dtype t, size_t raw_threshold_bytes,
                                      void* d_out, size_t out_capacity, uint64_t* d_out_offsets,
                                      void* d_workspace, size_t workspace_bytes, uint32_t* d_status,
                                      void* cuda_stream);

/* The send side of the exchange with the transfer fused into the encoder (PAPER.md L1361-1369:
 * Algorithm 4 lines 5 and 9, the row / column exchanges of compressed frontiers; L1792-1800, L1834: overlap of compression
 * and communication, the thesis's future work). As bfsc_compress_batch_codec, except that stream i is not appended to a
 * common output: it is written at the device address d_dst[i] — a device array of n_buf addresses, each a multiple of 16
 * with dst_capacity writable bytes behind it. An address may lie in ANOTHER GPU's memory (peer access enabled / an
 * NVLink-mapped symmetric buffer): the encoder's own stores are then the transfer, there is no packed send buffer, no
 * size exchange and no copy; the receiver finds the stream's size in its header (total_bytes, FORMAT.md §1) and decodes
 * its slots with bfsc_decompress_batch (d_in_offsets = the slots' offsets: a stream may be shorter than its span). The
 * bytes at d_dst[i] are identical to stream i of bfsc_compress_batch_codec. d_out_bytes[0..n_buf) (device, written):
 * total_bytes of each stream, 0 for a stream that did not fit dst_capacity (BFSC_ERR_DST_TOO_SMALL in *d_status; nothing
 * is written beyond a destination's capacity) or whose address is 0 or misaligned (BFSC_ERR_INVALID_ARG in *d_status).
 * Workspace: bfsc_workspace_bytes(total IDs, n_buf). Complete (visible to the owner of the destination) when the call's
 * last kernel has finished: order the receiver's decode behind it with an event, a stream-ordered collective or a
 * symmetric-memory barrier. BFSC_CODEC_FLAG_RAW_FALLBACK: BFSC_ERR_UNSUPPORTED as for every batch call. */
bfsc_status bfsc_compress_batch_scatter(bfsc_codec codec, const void* d_ids, const uint64_t* d_in_offsets, size_t n_buf,
                                        bfsc_dtype t, size_t raw_threshold_bytes,
                                        void* const* d_dst, size_t dst_capacity, uint64_t* d_out_bytes,
                                        void* d_workspace, size_t workspace_bytes, uint32_t* d_status,
                                        void* cuda_stream);

/* The receive side of the same exchange. d_in_offsets: n_buf+1 BYTE offsets
 * of the streams inside d_in (each a multiple of 16). IDs are written back to back at d_ids;
 * d_id_offsets[0..n_buf] (device, written) are their ELEMENT offsets. */
bfsc_status bfsc_decompress_batch(const void* d_in, const uint64_t* d_in_offsets, size_t n_buf,
                                  bfsc_dtype t,
                                  void* d_ids, size_t ids_capacity, uint64_t* d_id_offsets,
                                  void* d_workspace, size_t workspace_bytes, uint32_t* d_status,
                                  void* cuda_stream);

/* Frontier bitmaps (FORMAT.md §9; Algorithm 4 line 11, Algorithm 5): the codec fused
 * with the conversion on either side of it. d_bitmap: 32-bit words, bit v = bit v % 32 of word v / 32 <=> ID id_base + v;
 * 16-byte aligned, readable / writable up to a whole number of words.
 * bfsc_compress_bitmap: the stream of the ascending IDs of the set bits of d_bitmap[0 .. n_bits) — byte-identical to
 *   bfsc_compress_codec on that ID list, which is never materialised (the input read is n_bits / 8 bytes).
 *   out_capacity >= bfsc_compress_bound(number of set bits) (n_bits is always enough); workspace:
 *   bfsc_bitmap_workspace_bytes(n_bits, t).
 * bfsc_decompress_to_bitmap: ORs the bits of the stream's IDs into d_bitmap (old bits stay); *d_n_ids = IDs decoded.
 *   An ID outside [id_base, id_base + n_bits): BFSC_ERR_DST_TOO_SMALL in *d_status (bits of other IDs may have been set).
 * bfsc_decompress_to_frontier: Algorithm 4 lines 10-13 (t <- decompress(t''), t <- t (.) not Pi,
 *   Pi <- Pi + t, f <- t) in the decode kernel, with the next frontier and the visited set of Pi as two bitmaps of the
 *   same geometry: every decoded ID that is not in d_visited yet is set in d_visited and in d_frontier (both OR-ed:
 *   old bits stay); an ID that is visited already changes nothing. d_frontier != d_visited. Several calls of one BFS
 *   level (one per received stream) may run concurrently on the same pair of bitmaps: the updates are atomic and a
 *   vertex received twice enters the frontier once. Same error behaviour as bfsc_decompress_to_bitmap. */
size_t bfsc_bitmap_workspace_bytes(size_t n_bits, bfsc_dtype t);
bfsc_status bfsc_compress_bitmap(bfsc_codec codec, const uint32_t* d_bitmap, size_t n_bits, uint64_t id_base, bfsc_dtype t,
                                 size_t raw_threshold_bytes, void* d_out, size_t out_capacity, uint64_t* d_out_bytes,
                                 void* d_workspace, size_t workspace_bytes, uint32_t* d_status, void* cuda_stream);
bfsc_status bfsc_decompress_to_bitmap(const void* d_in, size_t in_bytes, bfsc_dtype t, uint64_t id_base,
                                      uint32_t* d_bitmap, size_t n_bits, uint64_t* d_n_ids,
                                      void* d_workspace, size_t workspace_bytes, uint32_t* d_status, void* cuda_stream);
bfsc_status bfsc_decompress_to_frontier(const void* d_in, size_t in_bytes, bfsc_dtype t, uint64_t id_base,
                                        uint32_t* d_frontier, uint32_t* d_visited, size_t n_bits, uint64_t* d_n_ids,
                                        void* d_workspace, size_t workspace_bytes, uint32_t* d_status, void* cuda_stream);

/* The receive side of a whole exchange in one call (Algorithm 4 lines 10-13 over all received streams, PAPER.md
 * L1369-1377): bfsc_decompress_to_frontier applied to the n_buf streams at d_in + d_in_offsets[i] (as in
 * bfsc_decompress_batch: byte offsets, multiples of 16, a stream may be shorter than its span — the slots of a receive
 * buffer). The result is the union: an ID that several streams carry, or that is visited already, enters the frontier
 * once or not at all, whatever the order. d_visited == NULL: no filter, every ID is OR-ed into d_frontier (the batch form
 * of bfsc_decompress_to_bitmap). *d_n_ids (device, written) = IDs decoded over all streams. Workspace:
 * bfsc_workspace_bytes(upper bound of the IDs of all streams together, n_buf); more blocks than it was sized for:
 * BFSC_ERR_INVALID_ARG in *d_status. At most 8192 streams (more: BFSC_ERR_UNSUPPORTED). Other errors as
 * bfsc_decompress_to_bitmap. */
bfsc_status bfsc_decompress_batch_to_frontier(const void* d_in, const uint64_t* d_in_offsets, size_t n_buf, bfsc_dtype t,
                                              uint64_t id_base, uint32_t* d_frontier, uint32_t* d_visited, size_t n_bits,
                                              uint64_t* d_n_ids, void* d_workspace, size_t workspace_bytes,
                                              uint32_t* d_status, void* cuda_stream);

/* Visited bitmaps (FORMAT.md §10; the predecessor / visited zone the
 * thesis left uncompressed, L2166: compressing the visited bitmap as future work). A bitmap of n_bits <= 2^32 bits (32-bit
 * words, bit v = bit v % 32 of word v / 32; bits >= n_bits of the last word are ignored) becomes a container that lists
 * its MINORITY bits — the set bits, or the clear bits of a mostly-visited bitmap — as one u32 stream of FORMAT.md §1, or
 * holds the bitmap itself when that would not be smaller: never more than bfsc_vbitmap_bound(n_bits) = 32 + the bitmap's
 * bytes rounded up to 16. Both calls: d_bitmap 4-byte aligned, d_out / d_in / d_workspace 16-byte aligned, workspace of
 * bfsc_vbitmap_workspace_bytes(n_bits) bytes (it holds a copy of the bitmap), stream-ordered, nothing allocated.
 * bfsc_compress_vbitmap: out_capacity >= bfsc_vbitmap_bound(n_bits) (else BFSC_ERR_DST_TOO_SMALL is returned);
 *   *d_out_bytes (device, written) = the container's total_bytes. codec = the rule of the stream inside.
 * bfsc_decompress_vbitmap: OVERWRITES d_bitmap[0 .. ceil(n_bits / 32)) (bits >= n_bits written as 0). n_bits must be the
 *   container's (else BFSC_ERR_DST_TOO_SMALL in *d_status); a malformed container or stream inside: BFSC_ERR_CORRUPT in
 *   *d_status; on either error d_bitmap is left as it was. */
size_t bfsc_vbitmap_bound(size_t n_bits);
size_t bfsc_vbitmap_workspace_bytes(size_t n_bits);
bfsc_status bfsc_compress_vbitmap(bfsc_codec codec, const uint32_t* d_bitmap, size_t n_bits, void* d_out, size_t out_capacity,
                                  uint64_t* d_out_bytes, void* d_workspace, size_t workspace_bytes, uint32_t* d_status,
                                  void* cuda_stream);
bfsc_status bfsc_decompress_vbitmap(const void* d_in, size_t in_bytes, uint32_t* d_bitmap, size_t n_bits,
                                    void* d_workspace, size_t workspace_bytes, uint32_t* d_status, void* cuda_stream);

/* End-to-end convenience calls with HOST buffers (pinned memory recommended): copy in,
 * run the device call above, copy the result out, synchronise the stream. d_scratch is a
 * caller-owned device buffer of at least bfsc_host_scratch_bytes(n_ids, t) bytes.
 * *h_out_bytes / *h_n_ids and the returned status include data-dependent errors. */
size_t bfsc_host_scratch_bytes(size_t n_ids, bfsc_dtype t);
bfsc_status bfsc_compress_host(const void* h_ids, size_t n_ids, bfsc_dtype t, size_t raw_threshold_bytes,
                               void* h_out, size_t out_capacity, uint64_t* h_out_bytes,
                               void* d_scratch, size_t scratch_bytes, void* cuda_stream);
bfsc_status bfsc_decompress_host(const void* h_in, size_t in_bytes, bfsc_dtype t,
                                 void* h_ids, size_t ids_capacity, uint64_t* h_n_ids,
                                 void* d_scratch, size_t scratch_bytes, void* cuda_stream);

/* Number of kernels the library has launched in this process so far (bench bookkeeping). */
uint64_t bfsc_kernel_launches(void);

#ifdef __cplusplus
}
#endif
#endif
