// decode.cu — bfsc_decompress / bfsc_decompress_batch (steps D0-D5).
//
// Launches per call, chained with programmatic dependent launch:
//   single stream                                   k_dec_tiles alone (it parses the stream header itself)
//   batch, small or of a few long streams           k_dec_tiles<..., kSelf> alone (every CTA plans for itself)
//   batch of up to 8192 streams                     k_dec_planblocks (from 3072 streams: k_dec_planchain) -> k_dec_tiles
//   larger batches                                  [k_dec_headers ->] k_dec_plan -> k_dec_blocks -> k_dec_tiles
//   into bitmaps (FORMAT.md §9)                     the same kernels with the bitmap sink (single stream and batches up to 8192 streams)
//   visited bitmap (FORMAT.md §10)                  k_vb_begin -> k_dec_tiles (bitmap sink, skipped for kind 0) -> k_vb_end
#include <cstdlib>
#include <atomic>
#include <mutex>

#include "block_decode.cuh"
#include "quad_decode.cuh"

namespace bfsc {

struct DecArgs {
    const unsigned char* in;
    const unsigned long long* in_off;   // n_buf+1 byte offsets, or nullptr (single stream, in_single bytes)
    unsigned long long in_single;
    uint32_t n_buf;
    void* ids;
    unsigned long long ids_cap;
    unsigned long long* id_off;         // n_buf+1 (batch, written) or nullptr
    unsigned long long* n_ids_out;      // single: *d_n_ids, or nullptr
    uint32_t* status;
    BitSink sink;                       // bfsc_decompress_to_bitmap: where the IDs' bits go (ids == nullptr then)
    WsView ws;                          // blk_first, fixed_prefix (= id offsets)
    const unsigned int* skip;           // single-stream calls, or nullptr: *skip != 0 (device) = nothing to decode, return at once (FORMAT.md §10: kind 0)
    unsigned long long plan_tag;        // k_dec_planchain: this call's tag (never 0 in its low 48 bits, unique per call in the process)
    uint32_t plan_grid;                 //   its CTAs (0: another plan ran): k_dec_tiles clears their states behind it
};

__device__ __forceinline__ unsigned long long s_begin(const DecArgs& a, uint32_t i) {
    return a.in_off ? a.in_off[i] : 0ull;
}
__device__ __forceinline__ unsigned long long s_avail(const DecArgs& a, uint32_t i) {
    return a.in_off ? a.in_off[i + 1] - a.in_off[i] : a.in_single;
}

// ---- D0 (batches of many streams), first part: the 32-byte stream headers, scattered over the input, are
// gathered into ws.blk_tab (32 B per stream; the block table is written later, by k_dec_blocks) by the whole
// GPU: the one-CTA plan kernel then reads them back to back. One SM cannot keep thousands of scattered
// sector reads in flight (4096 streams: the plan took 18 us, 11 of them waiting for headers).
constexpr uint32_t kHeaderGatherMin = 512;               // streams from which the gather pays for its launch
template <int W>
__global__ void __launch_bounds__(256) k_dec_headers(DecArgs a) {
    pdl_wait();                                          // the call before this one is complete (workspace, inputs)
    pdl_launch_dependents();
    for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < a.n_buf; i += gridDim.x * blockDim.x) {
        const unsigned long long beg = a.in_off[i], end = a.in_off[i + 1];
        uint4 h0 = make_uint4(0, 0, 0, 0), h1 = h0;
        if (!(beg & 15) && end >= beg && end - beg >= 32) {
            h0 = *reinterpret_cast<const uint4*>(a.in + beg);
            h1 = *reinterpret_cast<const uint4*>(a.in + beg + 16);
        }
        a.ws.blk_tab[2 * (size_t)i] = h0;
        a.ws.blk_tab[2 * (size_t)i + 1] = h1;
    }
}

// ---- D0: plan. Parse + validate every stream header; prefixes of IDs and blocks. ----------
template <int W, bool kCached>          // kCached: the headers come from ws.blk_tab (k_dec_headers)
__global__ void __launch_bounds__(1024) k_dec_plan(DecArgs a) {
    __shared__ Scan2 sm[33];
    __shared__ int bad;
    __shared__ HintQueue hq;
    constexpr unsigned long long E = W / 8;
    pdl_wait();                                          // the call before this one is complete (workspace, inputs)
    pdl_launch_dependents();
    if (threadIdx.x == 0) { bad = 0; hq.n = 0; }
    __syncthreads();
    Scan2 carry{0, 0};
    constexpr int kIpt = 4;                              // streams per thread and round: 4096 streams per block scan
    for (uint32_t i0 = 0; i0 < a.n_buf; i0 += blockDim.x * kIpt) {
        Scan2 v[kIpt], sum{0, 0};
        unsigned long long beg[kIpt], avail[kIpt];
        bool rd[kIpt];
        unsigned long long tot_bytes[kIpt];
        uint4 h0[kIpt], h1[kIpt];
#pragma unroll
        for (int u = 0; u < kIpt; u++) {                 // phase 1: extents (independent loads)
            const uint32_t i = i0 + threadIdx.x * kIpt + u;
            beg[u] = 0; avail[u] = 0; rd[u] = false;
            if (i < a.n_buf) {
                beg[u] = s_begin(a, i);
                const unsigned long long end = a.in_off ? a.in_off[i + 1] : a.in_single;
                avail[u] = end >= beg[u] ? end - beg[u] : 0;
                rd[u] = !(beg[u] & 15) && avail[u] >= 32;
            }
        }
#pragma unroll
        for (int u = 0; u < kIpt; u++) {                 // phase 2: all headers in flight at once
            h0[u] = h1[u] = make_uint4(0, 0, 0, 0);
            if (rd[u]) {
                if constexpr (kCached) {
                    const uint32_t i = i0 + threadIdx.x * kIpt + u;
                    h0[u] = __ldcg(a.ws.blk_tab + 2 * (size_t)i);
                    h1[u] = __ldcg(a.ws.blk_tab + 2 * (size_t)i + 1);
                } else {
                    h0[u] = *reinterpret_cast<const uint4*>(a.in + beg[u]);
                    h1[u] = *reinterpret_cast<const uint4*>(a.in + beg[u] + 16);
                }
            }
        }
#pragma unroll
        for (int u = 0; u < kIpt; u++) {                 // phase 3: validation (FORMAT.md §4)
            const uint32_t i = i0 + threadIdx.x * kIpt + u;
            v[u] = Scan2{0, 0};
            tot_bytes[u] = 0;
            if (i < a.n_buf) {
                bool ok = rd[u];
                if (ok) {
                    const uint32_t mode = (h0[u].y >> 16) & 0xffu;
                    const unsigned long long n = (unsigned long long)h0[u].w << 32 | h0[u].z;
                    const unsigned long long total = (unsigned long long)h1[u].y << 32 | h1[u].x;
                    const unsigned long long nb = h1[u].z;
                    if (h0[u].x != 0x43534642u || (h0[u].y & 0xffu) != 1u || ((h0[u].y >> 8) & 0xffu) != (uint32_t)W ||
                        mode > 2u || (h0[u].y >> 24) != 0u)                  // mode 2 (BP128-D1) decodes as mode 1: FORMAT.md §7
                        ok = false;
                    else if (total > avail[u] || (total & 15) || total < 32) ok = false;
                    else if (mode == 0) { if (nb != 0 || n > (total - 32) / E) ok = false; }
                    else if (nb != (n + kBlk - 1) / kBlk || 32ull + ((4ull * (nb + 1) + 15ull) & ~15ull) > total)   // (nb is 32 bits wide: n < 2^39)
                        ok = false;
                    if (ok) { v[u].a = nb; v[u].b = n; tot_bytes[u] = total; }
                }
                if (!ok) bad = 1;
            }
            sum.a += v[u].a; sum.b += v[u].b;
        }
        Scan2 tot;
        Scan2 ex = block_scan_excl2(sum, &tot, sm);
        ex.a += carry.a; ex.b += carry.b;
        // 16-byte stores of the thread's four table entries (see k_enc_plan); stream_start = the validated
        // total_bytes of the stream.
        const uint32_t ib = i0 + threadIdx.x * kIpt;
        unsigned long long bf[kIpt], fp[kIpt];
#pragma unroll
        for (int u = 0; u < kIpt; u++) {
            bf[u] = ex.a; fp[u] = ex.b;
            if (ib + u < a.n_buf) plan_hints_of(ib + u, ex.a, v[u].a, a.ws.tile_state, a.ws.tile_cap, &hq);
            ex.a += v[u].a; ex.b += v[u].b;
        }
        if (ib + kIpt <= a.n_buf) {
#pragma unroll
            for (int u = 0; u < kIpt; u += 2) {
                *reinterpret_cast<ulonglong2*>(a.ws.blk_first + ib + u) = make_ulonglong2(bf[u], bf[u + 1]);
                *reinterpret_cast<ulonglong2*>(a.ws.fixed_prefix + ib + u) = make_ulonglong2(fp[u], fp[u + 1]);
                *reinterpret_cast<ulonglong2*>(a.ws.stream_start + ib + u) = make_ulonglong2(tot_bytes[u], tot_bytes[u + 1]);
            }
        } else {
#pragma unroll
            for (int u = 0; u < kIpt; u++)
                if (ib + u < a.n_buf) { a.ws.blk_first[ib + u] = bf[u]; a.ws.fixed_prefix[ib + u] = fp[u]; a.ws.stream_start[ib + u] = tot_bytes[u]; }
        }
        carry.a += tot.a; carry.b += tot.b;
        plan_hints_flush(a.ws.tile_state, a.ws.tile_cap, &hq);
    }
    __syncthreads();
    const bool good = !bad && carry.a <= a.ws.blk_cap && carry.b <= a.ids_cap;
    if (threadIdx.x == 0) a.ws.blk_first[a.n_buf] = carry.a;
    if (threadIdx.x == 0) {
        a.ws.fixed_prefix[a.n_buf] = carry.b;
        a.ws.hdr->total_blocks = carry.a;
        a.ws.hdr->total_out = carry.b;
        a.ws.hdr->ok = good ? 1u : 0u;
        if (bad) set_status(a.status, BFSC_ERR_CORRUPT);
        else if (carry.b > a.ids_cap) set_status(a.status, BFSC_ERR_DST_TOO_SMALL);
        else if (!good) set_status(a.status, BFSC_ERR_INVALID_ARG);
        if (a.n_ids_out) *a.n_ids_out = good ? carry.b : 0ull;
    }
    __syncthreads();
    if (a.id_off)
        for (uint32_t i = threadIdx.x; i <= a.n_buf; i += blockDim.x) a.id_off[i] = good ? a.ws.fixed_prefix[i] : 0ull;
}

// ---- D0 (batch calls), second part: the block table. One thread per block of the batch: its stream
// (search from the group hint), which block of the stream it is and where its IDs go -> ws.blk_tab, so that
// k_dec_tiles reaches a block's directory entry with one load instead of a chain of dependent ones.
constexpr int kBlkTabThreads = 256;
template <int W>
__global__ void __launch_bounds__(kBlkTabThreads) k_dec_blocks(DecArgs a) {
    pdl_wait();
    pdl_launch_dependents();
    if (a.ws.hdr->ok == 0) return;
    const unsigned long long total = a.ws.hdr->total_blocks;
    for (unsigned long long g = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; g < total;
         g += (unsigned long long)gridDim.x * blockDim.x) {
        const uint32_t i = find_buf_from(a.ws.blk_first, a.n_buf, g, group_hint(a.ws.tile_state, g));
        const unsigned long long k = g - a.ws.blk_first[i], id0 = a.ws.fixed_prefix[i], n = a.ws.fixed_prefix[i + 1] - id0;
        const unsigned long long sb = s_begin(a, i), xi = id0 + kBlk * k;
        uint4 e0, e1;
        e0.x = (uint32_t)sb; e0.y = (uint32_t)(sb >> 32); e0.z = (uint32_t)xi; e0.w = (uint32_t)(xi >> 32);
        e1.x = (uint32_t)k; e1.y = (uint32_t)min((unsigned long long)kBlk, n - kBlk * k);
        e1.z = (uint32_t)(a.ws.stream_start[i] >> 4); e1.w = (uint32_t)((n + kBlk - 1) / kBlk);
        a.ws.blk_tab[2 * g] = e0; a.ws.blk_tab[2 * g + 1] = e1;
    }
}


// ---- D0 (batch calls of up to kFusedMaxStreams streams): plan AND block table in ONE launch of a few CTAs, as on the
// encode side (k_enc_planblocks): every CTA parses all the headers and scans for itself (no inter-CTA dependency, no
// gather / plan / table chain of three launches), keeps first block, first ID and size of every stream in shared
// memory, and writes its slice of the per-stream tables, of d_id_offsets and of the block table.
constexpr uint32_t kFusedMaxStreams = 8192;
constexpr int kFusedPlanCtas = 1024;                      // upper bound (a thread owns the table entries of the streams with i % grid == its CTA); the launch uses one CTA per SM: every CTA reads every header from L2 (148 CTAs x 4096 streams x 64 B = 39 MB), the block table is what is shared out (4096-buffer batch: 32 CTAs 42.4 us per decompress call, 74: 40.1, 148: 38.9)
__host__ __device__ inline size_t dec_planblocks_smem(size_t n_buf) { return 8 * (n_buf + 1) + 4 * (n_buf + 2) + 4 * (n_buf + 2); }
// The scan of both fused plans (any CTA size): headers of all streams parsed and validated (FORMAT.md §4), per stream
// first block, first ID and total_bytes / 16 -> shared memory; kTables: the per-stream workspace tables as well, the
// entries of the threads with `mine`. Returns the totals (blocks, IDs); *bad is set when a header is rejected.
template <int W, bool kTables>
__device__ __forceinline__ Scan2 dec_plan_scan(const DecArgs& a, unsigned long long* s_idpre, uint32_t* s_first, uint32_t* s_tot16,
                                               Scan2* sm, int* bad_p, bool mine) {
    constexpr unsigned long long E = W / 8;
    Scan2 carry{0, 0};
    constexpr int kIpt = 4;
    for (uint32_t i0 = 0; i0 < a.n_buf; i0 += blockDim.x * kIpt) {
        Scan2 v[kIpt], sum{0, 0};
        unsigned long long beg[kIpt], avail[kIpt], tot_bytes[kIpt];
        bool rd[kIpt];
        uint4 h0[kIpt], h1[kIpt];
#pragma unroll
        for (int u = 0; u < kIpt; u++) {                 // extents (independent loads)
            const uint32_t i = i0 + threadIdx.x * kIpt + u;
            beg[u] = 0; avail[u] = 0; rd[u] = false;
            if (i < a.n_buf) {
                beg[u] = a.in_off[i];
                const unsigned long long end = a.in_off[i + 1];
                avail[u] = end >= beg[u] ? end - beg[u] : 0;
                rd[u] = !(beg[u] & 15) && avail[u] >= 32;
            }
        }
#pragma unroll
        for (int u = 0; u < kIpt; u++) {                 // all headers in flight at once
            h0[u] = h1[u] = make_uint4(0, 0, 0, 0);
            if (rd[u]) {
                h0[u] = __ldcg(reinterpret_cast<const uint4*>(a.in + beg[u]));
                h1[u] = __ldcg(reinterpret_cast<const uint4*>(a.in + beg[u] + 16));
            }
        }
#pragma unroll
        for (int u = 0; u < kIpt; u++) {                 // validation (FORMAT.md §4), as in k_dec_plan
            const uint32_t i = i0 + threadIdx.x * kIpt + u;
            v[u] = Scan2{0, 0};
            tot_bytes[u] = 0;
            if (i < a.n_buf) {
                bool ok = rd[u];
                if (ok) {
                    const uint32_t mode = (h0[u].y >> 16) & 0xffu;
                    const unsigned long long n = (unsigned long long)h0[u].w << 32 | h0[u].z;
                    const unsigned long long total = (unsigned long long)h1[u].y << 32 | h1[u].x;
                    const unsigned long long nb = h1[u].z;
                    if (h0[u].x != 0x43534642u || (h0[u].y & 0xffu) != 1u || ((h0[u].y >> 8) & 0xffu) != (uint32_t)W ||
                        mode > 2u || (h0[u].y >> 24) != 0u)
                        ok = false;
                    else if (total > avail[u] || (total & 15) || total < 32) ok = false;
                    else if (mode == 0) { if (nb != 0 || n > (total - 32) / E) ok = false; }
                    else if (nb != (n + kBlk - 1) / kBlk || 32ull + ((4ull * (nb + 1) + 15ull) & ~15ull) > total)
                        ok = false;
                    if (ok) { v[u].a = nb; v[u].b = n; tot_bytes[u] = total; }
                }
                if (!ok) *bad_p = 1;
            }
            sum.a += v[u].a; sum.b += v[u].b;
        }
        Scan2 tot;
        Scan2 ex = block_scan_excl2(sum, &tot, sm);
        ex.a += carry.a; ex.b += carry.b;
#pragma unroll
        for (int u = 0; u < kIpt; u++) {
            const uint32_t i = i0 + threadIdx.x * kIpt + u;
            if (i < a.n_buf) {
                s_first[i] = (uint32_t)ex.a; s_idpre[i] = ex.b; s_tot16[i] = (uint32_t)(tot_bytes[u] >> 4);
                if (kTables && mine) { a.ws.blk_first[i] = ex.a; a.ws.fixed_prefix[i] = ex.b; a.ws.stream_start[i] = tot_bytes[u]; }
            }
            ex.a += v[u].a; ex.b += v[u].b;
        }
        carry.a += tot.a; carry.b += tot.b;
    }
    return carry;
}

template <int W>
__global__ void __launch_bounds__(1024) k_dec_planblocks(DecArgs a) {
    extern __shared__ __align__(16) unsigned char pb_smem[];
    unsigned long long* s_idpre = reinterpret_cast<unsigned long long*>(pb_smem);      // n_buf + 1: first ID of every stream
    uint32_t* s_first = reinterpret_cast<uint32_t*>(s_idpre + a.n_buf + 1);            // n_buf + 1: first block
    uint32_t* s_tot16 = s_first + a.n_buf + 2;                                         // n_buf: validated total_bytes / 16
    __shared__ Scan2 sm[33];
    __shared__ int bad;
    pdl_wait();                                          // the call before this one is complete (workspace, inputs)
    pdl_launch_dependents();
    if (threadIdx.x == 0) bad = 0;
    __syncthreads();
    const bool mine = threadIdx.x % gridDim.x == blockIdx.x;
    const Scan2 carry = dec_plan_scan<W, true>(a, s_idpre, s_first, s_tot16, sm, &bad, mine);
    if (threadIdx.x == 0) { s_first[a.n_buf] = (uint32_t)carry.a; s_idpre[a.n_buf] = carry.b; }
    __syncthreads();
    const bool good = !bad && carry.a <= a.ws.blk_cap && carry.b <= a.ids_cap && carry.a < (1ull << 32);
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        a.ws.blk_first[a.n_buf] = carry.a;
        a.ws.fixed_prefix[a.n_buf] = carry.b;
        a.ws.hdr->total_blocks = carry.a;
        a.ws.hdr->total_out = carry.b;
        a.ws.hdr->ok = good ? 1u : 0u;
        if (bad) set_status(a.status, BFSC_ERR_CORRUPT);
        else if (carry.b > a.ids_cap) set_status(a.status, BFSC_ERR_DST_TOO_SMALL);
        else if (!good) set_status(a.status, BFSC_ERR_INVALID_ARG);
        if (a.n_ids_out) *a.n_ids_out = good ? carry.b : 0ull;
    }
    const unsigned long long stride = (unsigned long long)gridDim.x * blockDim.x, me = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (a.id_off)
        for (unsigned long long i = me; i <= a.n_buf; i += stride) a.id_off[i] = good ? s_idpre[i] : 0ull;
    if (!good) return;
    for (unsigned long long g = me; g < carry.a; g += stride) {
        uint32_t lo = 0, hi = a.n_buf;                   // the last i with s_first[i] <= g
        while (hi - lo > 1) {
            const uint32_t mid = (lo + hi) >> 1;
            if (s_first[mid] <= (uint32_t)g) lo = mid; else hi = mid;
        }
        const uint32_t i = lo;
        const unsigned long long k = g - s_first[i], id0 = s_idpre[i], n = s_idpre[i + 1] - id0;
        const unsigned long long sb = a.in_off[i], xi = id0 + kBlk * k;
        uint4 e0, e1;
        e0.x = (uint32_t)sb; e0.y = (uint32_t)(sb >> 32); e0.z = (uint32_t)xi; e0.w = (uint32_t)(xi >> 32);
        e1.x = (uint32_t)k; e1.y = (uint32_t)min((unsigned long long)kBlk, n - kBlk * k);
        e1.z = s_tot16[i]; e1.w = (uint32_t)((n + kBlk - 1) / kBlk);
        a.ws.blk_tab[2 * g] = e0; a.ws.blk_tab[2 * g + 1] = e1;
    }
}

// ---- D0 for batches of MANY streams (kChainMinStreams .. kFusedMaxStreams): a single-pass CHAINED plan. The fused plan
// above lets every CTA parse every header (no inter-CTA dependency, right for a handful of streams); with thousands of
// streams that redundancy is the call's cost (4096 streams: 13.5 of 38.9 us). Here the streams are dealt out: a CTA takes
// a ticket, parses the headers of slice `ticket` (<= 256 streams, one per thread), scans them, publishes the slice's
// sums (blocks, IDs, rejected headers) and gets its prefix from the sums of the lower tickets — held by CTAs that
// arrived earlier, so a CTA only ever waits for CTAs that are running or done (no residency assumption). Then it writes
// the per-stream tables, d_id_offsets and the block-table entries of ITS OWN streams (a warp per stream, no search;
// streams of more than kChainBigBlocks blocks by the whole CTA). The CTA with the last ticket knows the totals and
// writes the verdict. States live in ws.tile_state (4 words per ticket: tag, blocks, IDs, rejected), the ticket counter
// in ws.hdr; both are valid only with this call's TAG (host-side counter, unique per call), so whatever the workspace
// held before reads as "not yet published"; k_dec_tiles clears them behind the plan so that a replay of a captured
// call — same tag again — starts clean.
constexpr uint32_t kChainMinStreams = 3072;                // measured, us per decompress call, chained / every-CTA-for-itself: 512 streams 18.0 / 13.3, 1024 19.9 / 16.4, 2048 24.7 / 23.2, 4096 35.9 / 38.9 (4096 short streams 23.6 / 26.7), 8192 34.6 / 48.6 — the chain pays seven dependent round trips (ticket, offsets, headers, publish, poll, payload, tables) where the other pays three
constexpr int kChainThreads = 256;
constexpr uint32_t kChainBigBlocks = 1024;
__device__ __forceinline__ unsigned long long dec_ld_volatile(const unsigned long long* p) {
    unsigned long long v;
    asm volatile("ld.volatile.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void dec_st_volatile(unsigned long long* p, unsigned long long v) {
    asm volatile("st.volatile.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}
template <int W>
__global__ void __launch_bounds__(kChainThreads) k_dec_planchain(DecArgs a) {
    constexpr unsigned long long E = W / 8;
    __shared__ Scan2 sm[33];
    __shared__ unsigned int s_ticket, s_nbig;
    __shared__ Scan2 s_base;
    __shared__ unsigned long long s_badbefore;
    __shared__ unsigned long long s_inoff[kChainThreads], s_id0[kChainThreads];
    __shared__ uint32_t s_nb[kChainThreads], s_tot16[kChainThreads], s_big[kChainThreads];
    __shared__ unsigned long long s_blk0[kChainThreads];
    pdl_wait();                                          // the call before this one is complete (workspace, inputs)
    pdl_launch_dependents();
    const unsigned long long tag48 = a.plan_tag & 0xffffffffffffull;
    if (threadIdx.x == 0) {
        // ticket word: (tag << 16 | tickets drawn); anything else = nobody has drawn yet. Whoever finds it without the
        // tag tries ONCE to install (tag << 16 | 0): if that fails somebody else has, and from then on the word only
        // moves through tagged values. Then one atomic add per CTA (a compare-and-swap loop of 148 contenders on one
        // word takes 148 rounds: 80 us).
        unsigned long long* tt = &a.ws.hdr->pad[0];
        const unsigned long long seen = dec_ld_volatile(tt);
        if ((seen >> 16) != tag48) atomicCAS(tt, seen, tag48 << 16);
        s_ticket = (unsigned int)(atomicAdd(tt, 1ull) & 0xffffull);
        s_nbig = 0;
    }
    __syncthreads();
    const uint32_t ticket = s_ticket, grid = gridDim.x;
    const uint32_t per = (a.n_buf + grid - 1) / grid;    // <= kChainThreads (the launch sees to it)
    const uint32_t lo = min(ticket * per, a.n_buf), hi = min(lo + per, a.n_buf);
    const uint32_t i = lo + threadIdx.x;
    // this thread's stream: header parsed and validated (FORMAT.md §4), as in dec_plan_scan
    Scan2 v{0, 0};
    unsigned long long beg = 0, tot_bytes = 0, bad = 0;
    if (i < hi) {
        beg = a.in_off[i];
        const unsigned long long end = a.in_off[i + 1];
        const unsigned long long avail = end >= beg ? end - beg : 0;
        bool ok = !(beg & 15) && avail >= 32;
        if (ok) {
            const uint4 h0 = __ldcg(reinterpret_cast<const uint4*>(a.in + beg));
            const uint4 h1 = __ldcg(reinterpret_cast<const uint4*>(a.in + beg + 16));
            const uint32_t mode = (h0.y >> 16) & 0xffu;
            const unsigned long long n = (unsigned long long)h0.w << 32 | h0.z;
            const unsigned long long total = (unsigned long long)h1.y << 32 | h1.x;
            const unsigned long long nb = h1.z;
            if (h0.x != 0x43534642u || (h0.y & 0xffu) != 1u || ((h0.y >> 8) & 0xffu) != (uint32_t)W || mode > 2u || (h0.y >> 24) != 0u)
                ok = false;
            else if (total > avail || (total & 15) || total < 32) ok = false;
            else if (mode == 0) { if (nb != 0 || n > (total - 32) / E) ok = false; }
            else if (nb != (n + kBlk - 1) / kBlk || 32ull + ((4ull * (nb + 1) + 15ull) & ~15ull) > total) ok = false;
            if (ok) { v.a = nb; v.b = n; tot_bytes = total; }
        }
        if (!ok) bad = 1;
    }
    const unsigned long long n_bad = __syncthreads_count(bad != 0);
    Scan2 tot;
    const Scan2 ex = block_scan_excl2(v, &tot, sm);
    unsigned long long* states = a.ws.tile_state;
    if (threadIdx.x == 0) {                              // publish: payload, fence, tag
        unsigned long long* st = states + 4ull * ticket;
        dec_st_volatile(st + 1, tot.a); dec_st_volatile(st + 2, tot.b); dec_st_volatile(st + 3, n_bad);
        __threadfence();
        dec_st_volatile(st, a.plan_tag);
    }
    if (threadIdx.x < 32) {
        // prefix over the lower tickets: first every tag this lane needs (independent polls), ONE fence, then the
        // payloads (independent loads) — a fence and two dependent round trips per state cost 8 us at 148 tickets
        constexpr int kMaxPer = 32;                      // states per lane: tickets < 1024
        Scan2 acc{0, 0};
        unsigned long long badb = 0;
        for (uint32_t j0 = threadIdx.x; j0 < ticket; j0 += 32 * kMaxPer) {
            uint32_t pending = 0;
#pragma unroll 1
            for (int u = 0; u < kMaxPer; u++)
                if (j0 + 32u * u < ticket) pending |= 1u << u;
            while (pending) {
                uint32_t still = 0;
                for (int u = 0; u < kMaxPer; u++)
                    if ((pending >> u & 1u) && dec_ld_volatile(states + 4ull * (j0 + 32u * u)) != a.plan_tag) still |= 1u << u;
                pending = still;
                if (pending) __nanosleep(64);
            }
        }
        __threadfence();
        for (uint32_t j = threadIdx.x; j < ticket; j += 32) {
            const unsigned long long* st = states + 4ull * j;
            acc.a += dec_ld_volatile(st + 1); acc.b += dec_ld_volatile(st + 2); badb += dec_ld_volatile(st + 3);
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            acc.a += __shfl_xor_sync(kFull, acc.a, o); acc.b += __shfl_xor_sync(kFull, acc.b, o); badb += __shfl_xor_sync(kFull, badb, o);
        }
        if (threadIdx.x == 0) { s_base = acc; s_badbefore = badb; }
    }
    __syncthreads();
    const Scan2 base = s_base;
    if (ticket == grid - 1 && threadIdx.x == 0) {        // the last ticket: totals and the verdict
        const unsigned long long blocks = base.a + tot.a, ids = base.b + tot.b;
        const bool any_bad = s_badbefore + n_bad != 0;
        const bool good = !any_bad && blocks <= a.ws.blk_cap && ids <= a.ids_cap && blocks < (1ull << 32);
        a.ws.blk_first[a.n_buf] = blocks;
        a.ws.fixed_prefix[a.n_buf] = ids;
        a.ws.hdr->total_blocks = blocks;
        a.ws.hdr->total_out = ids;
        a.ws.hdr->ok = good ? 1u : 0u;
        if (any_bad) set_status(a.status, BFSC_ERR_CORRUPT);
        else if (ids > a.ids_cap) set_status(a.status, BFSC_ERR_DST_TOO_SMALL);
        else if (!good) set_status(a.status, BFSC_ERR_INVALID_ARG);
        if (a.n_ids_out) *a.n_ids_out = good ? ids : 0ull;
        if (a.id_off) a.id_off[a.n_buf] = ids;           // (a rejected call: k_dec_tiles zeroes all of them)
    }
    // own streams: tables, d_id_offsets; block table by a warp per stream
    const unsigned long long blk0 = base.a + ex.a, id0 = base.b + ex.b;
    s_blk0[threadIdx.x] = blk0; s_id0[threadIdx.x] = id0; s_inoff[threadIdx.x] = beg;
    s_nb[threadIdx.x] = (uint32_t)min(v.a, 0xffffffffull); s_tot16[threadIdx.x] = (uint32_t)(tot_bytes >> 4);
    if (i < hi) {
        a.ws.blk_first[i] = blk0; a.ws.fixed_prefix[i] = id0; a.ws.stream_start[i] = tot_bytes;
        if (a.id_off) a.id_off[i] = id0;
        if (v.a > kChainBigBlocks) s_big[atomicAdd(&s_nbig, 1u)] = threadIdx.x;
    }
    __syncthreads();
    auto entry = [&](uint32_t t, unsigned long long k) {
        const unsigned long long g = s_blk0[t] + k;
        if (g >= a.ws.blk_cap) return;                   // (the call is rejected by the last ticket; nothing out of bounds)
        const unsigned long long nb = s_nb[t];
        // IDs of the stream: nb blocks, the last one ragged — from the header's n, kept as id0 of the next stream - id0
        const unsigned long long n = (t + 1 < hi - lo ? s_id0[t + 1] : base.b + tot.b) - s_id0[t];
        const unsigned long long sb = s_inoff[t], xi = s_id0[t] + kBlk * k;
        uint4 e0, e1;
        e0.x = (uint32_t)sb; e0.y = (uint32_t)(sb >> 32); e0.z = (uint32_t)xi; e0.w = (uint32_t)(xi >> 32);
        e1.x = (uint32_t)k; e1.y = (uint32_t)min((unsigned long long)kBlk, n - kBlk * k);
        e1.z = s_tot16[t]; e1.w = (uint32_t)nb;
        a.ws.blk_tab[2 * g] = e0; a.ws.blk_tab[2 * g + 1] = e1;
    };
    const uint32_t warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    for (uint32_t t = warp; t < hi - lo; t += kChainThreads / 32) {
        const uint32_t nb = s_nb[t];
        if (nb > kChainBigBlocks) continue;
        for (uint32_t k = lane; k < nb; k += 32) entry(t, k);
    }
    for (uint32_t b = 0; b < s_nbig; b++) {              // long streams: the whole CTA
        const uint32_t t = s_big[b];
        for (unsigned long long k = threadIdx.x; k < s_nb[t]; k += kChainThreads) entry(t, k);
    }
}

// ---- D1-D5 fused -------------------------------------------------------------------------
// Warp = batch of 8 consecutive blocks, four lanes per block (quad_decode.cuh). Per batch:
//   locate   per quad: stream, directory entries -> block address, span, valid IDs, output address
//   D1       cp.async the block (<= 336 B) into the warp's staging slots
//   D2-D4    unpack from shared memory, patch through the warp's table, scan, 128-bit stores
// Blocks over 336 B (b > 20: nearly incompressible data) take the warp-per-block path of
// block_decode.cuh, straight from global memory. Single-stream calls parse the stream header here
// (no plan kernel); RAW streams are copied at the end (D5).
// CTA shape: u32 2 CTAs of 16 warps per SM (6.9 KB of shared memory per warp), u64 2 CTAs of 8 warps (11 KB per warp);
// the TMA variant (two staging buffers per warp: 9.7 KB) fits 2 CTAs of 11 warps
template <int W, bool kTma = false> struct DecCfg {
    static constexpr int kStages = kTma ? 2 : 1;                                      // staging buffers per warp
    static constexpr int kWarps = (W == 32) ? (kTma ? 11 : 16) : 8;
    static constexpr int kThreads = kWarps * 32;
    static constexpr int kCtasPerSm = 2;
};

template <int W, bool kTma = false> struct DecSmem {
    using T = typename IdT<W>::T;
    static constexpr size_t kStageBytes = (size_t)DecCfg<W, kTma>::kStages * DecStage<W, kTma>::kStageChunks * 16;   // per warp
    static constexpr size_t kTabBytes = (size_t)kDecBlocks * kBlk * sizeof(T);         // per warp
    static constexpr size_t kBytes = DecCfg<W, kTma>::kWarps * (kStageBytes + kTabBytes);
};

template <int W>
struct BlockAt {                       // where the quad's block is
    const unsigned char* blk;          // first byte of the block (nullptr: no block / malformed)
    typename IdT<W>::T* x;             // first output ID
    uint32_t span16;                   // directory span in 16-byte units
    int m;                             // valid IDs
};

// kTma (single-stream calls): D1 as ONE bulk copy (TMA, cp.async.bulk + mbarrier) of the warp batch's contiguous span
// [dir[8k], dir[8k+8)) * 16 issued by lane 0, the blocks unpacked where they land; else every lane copies 16-byte
// chunks of its quad's block into the quad's slot (cp.async). The measured A/B is in DESIGN.md §5.2.
// kSelf (small batches: up to kSelfMaxStreams streams, kSelfMaxBlocks blocks): the whole call in ONE launch — every CTA
// runs D0 for itself (dec_plan_scan, tables in shared memory) instead of reading what a plan kernel left in the workspace.
constexpr uint32_t kSelfMaxStreams = 1024, kSelfMaxBlocks = 2048;
constexpr uint32_t kSelfFewStreams = 64, kSelfFewBlocks = 32768;   // a few long streams: kSelf up to so many blocks (no plan launch, no block table: 8 x 2^18 u32 IDs 10.3 -> 7.2 us per call; from ~10^5 blocks on the block table's single lookup per block wins: 64 x 220 K u64 IDs 37.3 / 40.7)
template <int W, bool kBatch, bool kTma, bool kBits = false, bool kSelf = false>   // kBatch: a.in_off != nullptr; kBits: bits into a.sink instead of IDs into a.ids
__global__ void __launch_bounds__(DecCfg<W, kTma>::kThreads, DecCfg<W, kTma>::kCtasPerSm) k_dec_tiles(DecArgs a) {
    static_assert(!kSelf || (kBatch && !kTma), "kSelf: batch calls");
    constexpr uint32_t kSelfN = kSelf ? kSelfMaxStreams : 0;
    __shared__ unsigned long long s_idpre[kSelfN + 1];                     // kSelf: first ID of every stream (entry n_buf: total)
    __shared__ uint32_t s_first[kSelfN + 2], s_tot16[kSelfN + 1];          //        first block, total_bytes / 16
    __shared__ Scan2 s_scan[kSelf ? 33 : 1];
    __shared__ int s_bad;
    constexpr int kDecWarps = DecCfg<W, kTma>::kWarps;
    using T = typename IdT<W>::T;
    constexpr unsigned long long E = W / 8;
    extern __shared__ __align__(16) unsigned char dec_smem[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, q = lane >> 2, l = lane & 3;
    uint4* stage = reinterpret_cast<uint4*>(dec_smem + warp * DecSmem<W, kTma>::kStageBytes);
    T* tab_w = reinterpret_cast<T*>(dec_smem + kDecWarps * DecSmem<W, kTma>::kStageBytes + warp * DecSmem<W, kTma>::kTabBytes);
    for (int x = lane; x < kDecBlocks * kBlk; x += 32) tab_w[x] = 0;       // patch table: all zero between uses
    __syncwarp();
    constexpr int kDecSpanMax = DecStage<W, kTma>::kSpanMax, kDecSlotChunks = DecStage<W, kTma>::kSlotChunks, kDecStageChunks = DecStage<W, kTma>::kStageChunks;
    uint4* slot = stage + kDecSlotChunks * q;
    T* tab = tab_w + kBlk * q;
    __shared__ unsigned long long s_mbar[kTma ? 2 * kDecWarps : 1];       // kTma: "the span in stage s of warp w has landed"
    if constexpr (kTma) {
        if (lane < 2) dec_mbar_init(&s_mbar[2 * warp + lane], 1);
        dec_fence_mbar_init();
        __syncwarp();
    }

    constexpr bool batch = kBatch;
    unsigned long long total_blocks, n1 = 0, total16_1 = 0, lo16_1 = 0;   // single stream: n, total/16, first block/16
    pdl_wait();                                                            // the kernel before this one is complete
    pdl_launch_dependents();                                               // the next one may be set up; it waits for this grid
    if constexpr (kSelf) {                                                 // D0 of the batch, by every CTA for itself
        if (threadIdx.x == 0) s_bad = 0;
        __syncthreads();
        const Scan2 tot = dec_plan_scan<W, false>(a, s_idpre, s_first, s_tot16, s_scan, &s_bad, false);
        if (threadIdx.x == 0) { s_first[a.n_buf] = (uint32_t)tot.a; s_idpre[a.n_buf] = tot.b; }
        __syncthreads();
        const bool good = !s_bad && tot.b <= a.ids_cap && tot.a < (1ull << 32);
        if (blockIdx.x == 0 && threadIdx.x == 0) {
            if (s_bad) set_status(a.status, BFSC_ERR_CORRUPT);
            else if (tot.b > a.ids_cap) set_status(a.status, BFSC_ERR_DST_TOO_SMALL);
            else if (!good) set_status(a.status, BFSC_ERR_INVALID_ARG);
            if (a.n_ids_out) *a.n_ids_out = good ? tot.b : 0ull;
        }
        if (a.id_off)
            for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i <= a.n_buf; i += gridDim.x * blockDim.x)
                a.id_off[i] = good ? s_idpre[i] : 0ull;
        if (!good) return;
        total_blocks = tot.a;
    } else if (batch) {
        if (a.plan_grid != 0 && blockIdx.x == 0) {                         // k_dec_planchain's states and ticket: cleared behind it
            for (uint32_t x = threadIdx.x; x < 4u * a.plan_grid; x += blockDim.x) a.ws.tile_state[x] = 0ull;
            if (threadIdx.x == 0) a.ws.hdr->pad[0] = 0ull;
        }
        if (!a.ws.hdr->ok) {
            if (a.plan_grid != 0 && a.id_off)                              // (the chained plan wrote them before the verdict was known)
                for (unsigned long long i = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; i <= a.n_buf; i += (unsigned long long)gridDim.x * blockDim.x)
                    a.id_off[i] = 0ull;
            return;
        }
        total_blocks = a.ws.hdr->total_blocks;
    } else {                                                               // D0 for one stream (FORMAT.md §1, §4)
        if (a.skip != nullptr && *a.skip != 0u) return;
        const bool first = blockIdx.x == 0 && threadIdx.x == 0;
        bool ok = a.in_single >= 32;
        uint32_t mode = 0;
        unsigned long long total = 0, nb = 0;
        if (ok) {
            const uint4 h0 = *reinterpret_cast<const uint4*>(a.in);
            const uint4 h1 = *reinterpret_cast<const uint4*>(a.in + 16);
            mode = (h0.y >> 16) & 0xffu;
            n1 = (unsigned long long)h0.w << 32 | h0.z;
            total = (unsigned long long)h1.y << 32 | h1.x;
            nb = h1.z;
            if (h0.x != 0x43534642u || (h0.y & 0xffu) != 1u || ((h0.y >> 8) & 0xffu) != (uint32_t)W || mode > 2u ||
                (h0.y >> 24) != 0u)
                ok = false;
            else if (total > a.in_single || (total & 15) || total < 32) ok = false;
            else if (mode == 0) { if (nb != 0 || n1 > (total - 32) / E) ok = false; }
            else if (nb != (n1 + kBlk - 1) / kBlk || 32ull + ((4ull * (nb + 1) + 15ull) & ~15ull) > total)
                ok = false;
        }
        if (!ok || n1 > a.ids_cap) {
            if (first) {
                set_status(a.status, ok ? BFSC_ERR_DST_TOO_SMALL : BFSC_ERR_CORRUPT);
                if (a.n_ids_out) *a.n_ids_out = 0;
            }
            return;
        }
        if (first && a.n_ids_out) *a.n_ids_out = n1;
        if (mode == 0) {                                                   // D5: raw passthrough
            const T* xs = reinterpret_cast<const T*>(a.in + 32);
            T* y = reinterpret_cast<T*>(a.ids);
            for (unsigned long long t = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; t < n1;
                 t += (unsigned long long)gridDim.x * blockDim.x)
                if constexpr (kBits) set_bits4<T>(a.sink, xs[t], (T)0, (T)0, (T)0, 1);
                else y[t] = xs[t];
            return;
        }
        total_blocks = nb;
        total16_1 = total >> 4;
        lo16_1 = (32ull + ((4ull * (nb + 1) + 15ull) & ~15ull)) >> 4;
    }

    uint32_t self_hint = 0;                                                // kSelf: the stream of this lane's last block
    auto locate = [&](unsigned long long g) -> BlockAt<W> {
        BlockAt<W> r; r.blk = nullptr; r.x = nullptr; r.span16 = 0; r.m = 0;
        if (g >= total_blocks) return r;
        const unsigned char* s = a.in;
        unsigned long long k = g, id0 = 0, n = n1, total16 = total16_1, lo16 = lo16_1;
        int m;
        unsigned long long xi;
        if constexpr (kSelf) {                                             // the CTA's own tables
            // the last i with s_first[i] <= g, searched from the stream of this lane's previous block (a warp's batches
            // ascend): gallop, then bisect — a level of a few long streams finds its stream with two reads
            uint32_t lo = s_first[self_hint] <= (uint32_t)g ? self_hint : 0u, step = 1;
            while (lo + step < a.n_buf && s_first[lo + step] <= (uint32_t)g) { lo += step; step <<= 1; }
            uint32_t hi = min(lo + step, a.n_buf);
            while (hi - lo > 1) {
                const uint32_t mid = (lo + hi) >> 1;
                if (s_first[mid] <= (uint32_t)g) lo = mid; else hi = mid;
            }
            self_hint = lo;
            s = a.in + a.in_off[lo];
            k = g - s_first[lo]; id0 = s_idpre[lo]; n = s_idpre[lo + 1] - id0; total16 = s_tot16[lo];
            m = (int)min((unsigned long long)kBlk, n - kBlk * k);
            xi = id0 + kBlk * k;
            lo16 = (32ull + ((4ull * ((n + kBlk - 1) / kBlk + 1) + 15ull) & ~15ull)) >> 4;
        } else if (batch) {                                                // ws.blk_tab, written by k_dec_blocks / k_dec_planblocks
            const uint4 e0 = __ldcg(a.ws.blk_tab + 2 * g), e1 = __ldcg(a.ws.blk_tab + 2 * g + 1);
            s = a.in + ((unsigned long long)e0.y << 32 | e0.x);
            xi = (unsigned long long)e0.w << 32 | e0.z;
            k = e1.x; m = (int)e1.y; total16 = e1.z;
            lo16 = (32ull + ((4ull * ((unsigned long long)e1.w + 1) + 15ull) & ~15ull)) >> 4;
        } else {
            m = (int)min((unsigned long long)kBlk, n - kBlk * k);
            xi = id0 + kBlk * k;
        }
        const uint32_t* dir = reinterpret_cast<const uint32_t*>(s + 32);
        const unsigned long long o0 = dir[k], o1 = dir[k + 1];
        if (o0 < lo16 || o1 <= o0 || o1 > total16) { set_status(a.status, BFSC_ERR_CORRUPT); return r; }
        r.blk = s + 16ull * o0;
        r.span16 = (uint32_t)(o1 - o0);
        r.m = m;
        r.x = reinterpret_cast<T*>(a.ids) + xi;
        BFSC_CHECK(kBits || xi + (unsigned long long)m <= a.ids_cap);
        return r;
    };

    const unsigned long long n_batches = (total_blocks + kDecBlocks - 1) / kDecBlocks;
    // Every working warp gets the same number of batches: with R = rounds the grid's warps need, only
    // ceil(n_batches / R) warps work, spread evenly over the CTAs (CTA c has base or base + 1 working warps,
    // numbered consecutively: neighbouring batches, i.e. neighbouring bytes of the stream, stay on one SM).
    // 2^24 IDs = 16384 batches on 296 x 16 warps: 4 rounds, 4096 warps with 4 batches each instead of 4736 with 3 or 4.
    const uint32_t cap_warps = gridDim.x * kDecWarps;
    unsigned long long n_warps = cap_warps;
    unsigned long long bi = (unsigned long long)blockIdx.x * kDecWarps + warp;
    if (n_batches > cap_warps && n_batches < 0xffffffffull) {             // (32-bit arithmetic: 64-bit divisions cost more than they save)
        const uint32_t nb32 = (uint32_t)n_batches, rounds = (nb32 + cap_warps - 1) / cap_warps;
        const uint32_t nw = (nb32 + rounds - 1) / rounds, base_w = nw / gridDim.x, rem_w = nw - base_w * gridDim.x;
        n_warps = nw;
        bi = blockIdx.x * base_w + min(blockIdx.x, rem_w) + warp;
        if ((uint32_t)warp >= base_w + (blockIdx.x < rem_w ? 1u : 0u)) bi = n_batches;   // this warp sits the call out
    }
    // D2-D4 of the quad's block, staged at `slot` (header chunk first)
    auto decode_staged = [&](const BlockAt<W>& cur, uint4* slot) {
        bool live = cur.blk != nullptr;
        const uint4 h = slot[0];
        const uint32_t b = h.z & 0xffu, n_exc = (h.z >> 8) & 0xffu;
        if (live && (b > (uint32_t)W || n_exc > 127u || 1u + b + exc_bytes<W>(n_exc) / 16u > cur.span16)) {
            set_status(a.status, BFSC_ERR_CORRUPT);
            live = false;
        }
        const unsigned char* e = reinterpret_cast<const unsigned char*>(slot + 1 + b);
        const bool patch = __any_sync(kFull, live && n_exc > 0);         // D3: scatter into the patch table
        if (patch) {
            if (!quad_patch_scatter<W>(tab, e, b, live ? n_exc : 0u, l)) { set_status(a.status, BFSC_ERR_CORRUPT); live = false; }
            __syncwarp();
            const int lv = live;                                     // all four shuffles by every lane: no short-circuit
            live = (__shfl_sync(kFull, lv, 4 * q + 0) & __shfl_sync(kFull, lv, 4 * q + 1) &
                    __shfl_sync(kFull, lv, 4 * q + 2) & __shfl_sync(kFull, lv, 4 * q + 3)) != 0;
        }
        const T base = (T)((unsigned long long)h.y << 32 | h.x);
        quad_decode_rows<W, kBatch, kBits>(slot + 1, live ? b : 0u, tab, patch, base, cur.x, live ? cur.m : 0, l, a.sink);   // D2-D4
        if (patch) {
            __syncwarp();
            quad_patch_clear<W>(tab, e, (cur.blk != nullptr && b <= (uint32_t)W && n_exc <= 127u && 1u + b + exc_bytes<W>(n_exc) / 16u <= cur.span16) ? n_exc : 0u, l);
        }
    };
    // slow path: the batch's blocks one at a time, the whole warp on each, straight from global memory
    auto decode_direct = [&](const BlockAt<W>& cur) {
        // slow path: one block at a time, the whole warp on it, straight from global memory
        for (int qq = 0; qq < kDecBlocks; qq++) {
            const unsigned char* blk = reinterpret_cast<const unsigned char*>(
                __shfl_sync(kFull, (unsigned long long)reinterpret_cast<uintptr_t>(cur.blk), 4 * qq));
            T* x = reinterpret_cast<T*>(__shfl_sync(kFull, (unsigned long long)reinterpret_cast<uintptr_t>(cur.x), 4 * qq));
            const uint32_t span16 = __shfl_sync(kFull, cur.span16, 4 * qq);
            const int m = __shfl_sync(kFull, cur.m, 4 * qq);
            if (blk == nullptr) continue;
            const uint4 h = *reinterpret_cast<const uint4*>(blk);
            const uint32_t b = h.z & 0xffu, n_exc = (h.z >> 8) & 0xffu;
            if (b > (uint32_t)W || n_exc > 127u || 16ull + 16ull * b + exc_bytes<W>(n_exc) > 16ull * span16) {
                set_status(a.status, BFSC_ERR_CORRUPT);
                continue;
            }
            const T base = (T)((unsigned long long)h.y << 32 | h.x);
            T dd[4];
            unpack_rows<W>(reinterpret_cast<const uint4*>(blk + 16), b, dd);
            if (n_exc > 0 && !patch_rows<W>(blk + 16 + 16 * b, b, n_exc, dd)) {
                set_status(a.status, BFSC_ERR_CORRUPT);
                continue;
            }
            scan_store<W, kBits>(dd, base, x, m, a.sink);
        }
    };

    if constexpr (!kTma) {
        BlockAt<W> cur = locate(bi * kDecBlocks + q);
        for (; bi < n_batches; bi += n_warps) {
            const bool big = cur.blk != nullptr && cur.span16 > (uint32_t)kDecSpanMax;
            const bool any_big = __any_sync(kFull, big);
            BFSC_CHECK(any_big || cur.blk == nullptr || cur.span16 <= (uint32_t)kDecSpanMax);
            if (!any_big && cur.blk != nullptr) quad_stage_block<kDecSpanMax>(slot, cur.blk, cur.span16, l);
            const BlockAt<W> nxt = locate((bi + n_warps) * kDecBlocks + q);   // the next batch's directory reads overlap the copy
            if (!any_big) {
                dec_cp_async_wait_all();
                __syncwarp();
                decode_staged(cur, slot);
                __syncwarp();                                                // slots and table free again
            } else {
                decode_direct(cur);
            }
            cur = nxt;
        }
    } else {
        // Two stages per warp: while batch i is unpacked from one, the span of batch i + 1 lands in the other — ONE bulk
        // copy (TMA) per batch, issued by lane 0: the batch's blocks are one contiguous piece of the stream (entry k + 1
        // of the directory ends block k and starts block k + 1). A quad whose directory entries were rejected breaks
        // the span: nothing of that batch is decoded (the status word says CORRUPT already).
        struct Staged { uint32_t rel; bool direct; bool skip; };
        auto issue = [&](BlockAt<W>& c, unsigned long long batch_i, int st) -> Staged {
            Staged r{0u, false, true};
            if (batch_i >= n_batches) return r;
            const bool expect = batch_i * kDecBlocks + q < total_blocks;
            const bool whole = __all_sync(kFull, !expect || c.blk != nullptr);
            const bool any_big = __any_sync(kFull, c.blk != nullptr && c.span16 > (uint32_t)kDecSpanMax);
            const unsigned long long base_p = __shfl_sync(kFull, (unsigned long long)reinterpret_cast<uintptr_t>(c.blk), 0);
            const int n_live = __popc(__ballot_sync(kFull, expect)) >> 2;
            r.rel = c.blk != nullptr ? (uint32_t)((reinterpret_cast<uintptr_t>(c.blk) - base_p) >> 4) : 0u;
            const uint32_t span_all = __shfl_sync(kFull, r.rel + c.span16, 4 * (n_live > 0 ? n_live - 1 : 0));
            if (!whole) { c.blk = nullptr; return r; }
            r.skip = false;
            r.direct = any_big;
            if (!any_big && lane == 0) {
                dec_mbar_expect_tx(&s_mbar[2 * warp + st], 16u * span_all);
                dec_bulk_load(stage + st * kDecStageChunks, reinterpret_cast<const void*>(static_cast<uintptr_t>(base_p)), 16u * span_all,
                              &s_mbar[2 * warp + st]);
            }
            return r;
        };
        BlockAt<W> cur = locate(bi * kDecBlocks + q);
        Staged sc = issue(cur, bi, 0);
        BlockAt<W> nxt = locate((bi + n_warps) * kDecBlocks + q);
        uint32_t phase[2] = {0u, 0u};
        int st = 0;
        for (; bi < n_batches; bi += n_warps) {
            const Staged sn = issue(nxt, bi + n_warps, st ^ 1);                  // lands while this batch is unpacked
            const BlockAt<W> nxt2 = locate((bi + 2 * n_warps) * kDecBlocks + q); // directory reads two batches ahead
            if (!sc.skip) {
                if (!sc.direct) {
                    dec_mbar_wait(&s_mbar[2 * warp + st], phase[st]);
                    phase[st] ^= 1u;
                    decode_staged(cur, stage + st * kDecStageChunks + sc.rel);
                    __syncwarp();                                            // stage and table free again
                } else {
                    decode_direct(cur);
                }
            }
            cur = nxt; nxt = nxt2; sc = sn; st ^= 1;
        }
    }

    if (batch) {                                                           // D5: raw streams of the batch
        for (uint32_t i = blockIdx.x; i < a.n_buf; i += gridDim.x) {
            const unsigned char* s = a.in + s_begin(a, i);
            if (s[6] != 0) continue;
            unsigned long long id0, n;
            if constexpr (kSelf) { id0 = s_idpre[i]; n = s_idpre[i + 1] - id0; }
            else { id0 = a.ws.fixed_prefix[i]; n = a.ws.fixed_prefix[i + 1] - id0; }
            const T* xs = reinterpret_cast<const T*>(s + 32);
            if constexpr (kBits) {
                for (unsigned long long t = threadIdx.x; t < n; t += blockDim.x) set_bits4<T>(a.sink, xs[t], (T)0, (T)0, (T)0, 1);
            } else {
                T* y = reinterpret_cast<T*>(a.ids) + id0;
                for (unsigned long long t = threadIdx.x; t < n; t += blockDim.x) y[t] = xs[t];
            }
        }
    }
}

// Once per device and instantiation: the dynamic shared memory attribute and the resident CTAs per SM.
template <int W, bool kBatch, bool kTma, bool kBits = false, bool kSelf = false>
static int dec_ctas_per_sm(int device) {
    static std::mutex mu;
    static int per_sm[kMaxDevices] = {};
    std::lock_guard<std::mutex> lock(mu);
    if (per_sm[device] == 0) {
        int n = 0;
        if (cudaFuncSetAttribute(k_dec_tiles<W, kBatch, kTma, kBits, kSelf>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)DecSmem<W, kTma>::kBytes) != cudaSuccess)
            return 0;
        if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, k_dec_tiles<W, kBatch, kTma, kBits, kSelf>, DecCfg<W, kTma>::kThreads, DecSmem<W, kTma>::kBytes) != cudaSuccess || n < 1)
            return 0;
        per_sm[device] = n;
    }
    return per_sm[device];
}

template <int W>
static bool dec_planblocks_init(int device) {            // once per device: the fused plan's shared memory (up to 128 KB)
    static std::mutex mu;
    static bool done[kMaxDevices] = {};
    std::lock_guard<std::mutex> lock(mu);
    if (!done[device]) {
        if (cudaFuncSetAttribute(k_dec_planblocks<W>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                 (int)dec_planblocks_smem(kFusedMaxStreams)) != cudaSuccess)
            return false;
        done[device] = true;
    }
    return true;
}

static unsigned long long next_plan_tag() {              // unique per call in the process, low 48 bits never 0
    static std::atomic<unsigned long long> counter{0x5bf5c0de0001ull};
    unsigned long long t;
    do { t = counter.fetch_add(1ull) + 1ull; } while ((t & 0xffffffffffffull) == 0);
    return t;
}

template <int W>
static bfsc_status launch_decode(const DecArgs& a_in, size_t max_blocks, cudaStream_t s) {
    DecArgs a = a_in;
    a.plan_tag = 0; a.plan_grid = 0;
    constexpr size_t kSmem = DecSmem<W>::kBytes;
    DeviceInfo dev;
    if (!current_device(&dev)) return BFSC_ERR_CUDA;
    // D1 staging of single-stream calls: per-lane cp.async (default) or, with BFSC_DEC_STAGING=tma in the environment,
    // one bulk copy (TMA) per warp batch into a two-stage ring. Both are bit-exact (tests run both); the measured
    // A/B (profiles/r2_dec_staging_ab.md) is why cp.async is the default.
    const char* staging = getenv("BFSC_DEC_STAGING");
    const bool use_tma = staging != nullptr && staging[0] == 't';
    const int per_sm = a.in_off ? dec_ctas_per_sm<W, true, false>(dev.device)
                                : (use_tma ? dec_ctas_per_sm<W, false, true>(dev.device) : dec_ctas_per_sm<W, false, false>(dev.device));
    if (per_sm < 1) return BFSC_ERR_CUDA;
    const int max_grid = dev.sms * per_sm;
    const int warps = a.in_off || !use_tma ? DecCfg<W, false>::kWarps : DecCfg<W, true>::kWarps;
    if (a.in_off && a.ws.blk_cap < max_blocks) max_blocks = a.ws.blk_cap;          // (more blocks than that: INVALID_ARG on the device)
    // CTAs: one per warp batch while the device has room for them (a small call is spread over the SMs, one working
    // warp each: k_dec_tiles balances the working warps over the CTAs), at most one resident wave
    (void)warps;
    const size_t want = (max_blocks + kDecBlocks - 1) / kDecBlocks;
    int grid = want < (size_t)max_grid ? (int)want : max_grid;
    if (grid < 1) grid = 1;
    const bool bits = a.sink.bm != nullptr;                                        // IDs -> bits of a frontier bitmap
    if (a.in_off && a.n_buf <= kSelfMaxStreams && (max_blocks <= kSelfMaxBlocks || (a.n_buf <= kSelfFewStreams && max_blocks <= kSelfFewBlocks))) {
        // a small batch (both bounds known on the host: stream count, and blocks by the ID capacity / the workspace size):
        // one launch, no plan kernel
        const int psm = bits ? dec_ctas_per_sm<W, true, false, true, true>(dev.device) : dec_ctas_per_sm<W, true, false, false, true>(dev.device);
        if (psm < 1) return BFSC_ERR_CUDA;
        const int g = want < (size_t)(dev.sms * psm) ? (want ? (int)want : 1) : dev.sms * psm;
        if (bits) BFSC_LAUNCH(launch_dep(k_dec_tiles<W, true, false, true, true>, g, DecCfg<W>::kThreads, kSmem, s, a));
        else BFSC_LAUNCH(launch_dep(k_dec_tiles<W, true, false, false, true>, g, DecCfg<W>::kThreads, kSmem, s, a));
    } else if (a.in_off && a.n_buf <= kFusedMaxStreams && a.ws.blk_cap < (1ull << 32)) {
        if (!dec_planblocks_init<W>(dev.device)) return BFSC_ERR_CUDA;
        if (bits && dec_ctas_per_sm<W, true, false, true>(dev.device) < 1) return BFSC_ERR_CUDA;
        // many streams: the chained plan (streams dealt out over the CTAs, 4 state words per CTA in ws.tile_state);
        // few: the plan every CTA runs for itself
        size_t cgrid = (size_t)dev.sms;
        if (cgrid > 2 * a.ws.tile_cap) cgrid = 2 * a.ws.tile_cap;
        if (cgrid > 0xffffu) cgrid = 0xffffu;
        if (a.n_buf >= kChainMinStreams && cgrid >= 1 && (a.n_buf + cgrid - 1) / cgrid <= (size_t)kChainThreads) {
            a.plan_tag = next_plan_tag(); a.plan_grid = (uint32_t)cgrid;
            BFSC_LAUNCH(launch_dep(k_dec_planchain<W>, (int)cgrid, kChainThreads, 0, s, a));
        } else {
            size_t pgrid = (a.ws.blk_cap + 1023) / 1024;
            if (pgrid > (size_t)dev.sms) pgrid = (size_t)dev.sms;
            if (pgrid > (size_t)kFusedPlanCtas) pgrid = kFusedPlanCtas;
            BFSC_LAUNCH(launch_dep(k_dec_planblocks<W>, pgrid ? (int)pgrid : 1, 1024, dec_planblocks_smem(a.n_buf), s, a));
        }
        if (bits) BFSC_LAUNCH(launch_dep(k_dec_tiles<W, true, false, true>, grid, DecCfg<W>::kThreads, kSmem, s, a));
        else BFSC_LAUNCH(launch_dep(k_dec_tiles<W, true, false>, grid, DecCfg<W>::kThreads, kSmem, s, a));
    } else if (a.in_off && bits) {
        return BFSC_ERR_UNSUPPORTED;                                               // (more than kFusedMaxStreams streams into a bitmap)
    } else if (a.in_off) {
        const bool gather = a.n_buf >= kHeaderGatherMin && a.ws.blk_cap >= a.n_buf;
        if (gather) {
            int hgrid = (int)((a.n_buf + 255) / 256);
            if (hgrid > dev.sms * 4) hgrid = dev.sms * 4;
            BFSC_LAUNCH(launch_dep(k_dec_headers<W>, hgrid, 256, 0, s, a));
        }
        if (gather) BFSC_LAUNCH(launch_dep(k_dec_plan<W, true>, 1, 1024, 0, s, a));
        else BFSC_LAUNCH(launch_dep(k_dec_plan<W, false>, 1, 1024, 0, s, a));
        size_t bgrid = (a.ws.blk_cap + kBlkTabThreads - 1) / kBlkTabThreads;
        if (bgrid > (size_t)dev.sms * 8) bgrid = (size_t)dev.sms * 8;
        BFSC_LAUNCH(launch_dep(k_dec_blocks<W>, bgrid ? (int)bgrid : 1, kBlkTabThreads, 0, s, a));
        BFSC_LAUNCH(launch_dep(k_dec_tiles<W, true, false>, max_grid, DecCfg<W>::kThreads, kSmem, s, a));
    } else if (a.sink.bm != nullptr) {
        const int psm = dec_ctas_per_sm<W, false, false, true>(dev.device);
        if (psm < 1) return BFSC_ERR_CUDA;
        const int g = want < (size_t)(dev.sms * psm) ? (want ? (int)want : 1) : dev.sms * psm;
        BFSC_LAUNCH(launch_dep(k_dec_tiles<W, false, false, true>, g, DecCfg<W>::kThreads, kSmem, s, a));
    } else {
        if (use_tma) BFSC_LAUNCH(launch_dep(k_dec_tiles<W, false, true>, grid, DecCfg<W, true>::kThreads, DecSmem<W, true>::kBytes, s, a));
        else BFSC_LAUNCH(launch_dep(k_dec_tiles<W, false, false>, grid, DecCfg<W>::kThreads, kSmem, s, a));
    }
    return BFSC_OK;
}

static bfsc_status decode_common(const void* d_in, const uint64_t* d_in_off, size_t in_single, size_t n_buf,
                                 bfsc_dtype t, void* d_ids, size_t ids_cap, uint64_t* d_id_off, uint64_t* d_n_ids,
                                 void* ws, size_t ws_bytes, uint32_t* d_status, void* stream,
                                 BitSink sink = BitSink{nullptr, 0, 0, nullptr, nullptr}, const unsigned int* skip = nullptr) {
    if (t != BFSC_U32 && t != BFSC_U64) return BFSC_ERR_INVALID_ARG;
    if (!d_in || !ws || n_buf > 0x7fffffffu) return BFSC_ERR_INVALID_ARG;
    if (!d_ids && ids_cap && !sink.bm) return BFSC_ERR_INVALID_ARG;
    if (((uintptr_t)d_in & 15) || ((uintptr_t)d_ids & 15) || ((uintptr_t)ws & 15)) return BFSC_ERR_INVALID_ARG;
    DecArgs a;
    if (!ws_carve(ws, ws_bytes, n_buf, &a.ws)) return BFSC_ERR_INVALID_ARG;
    a.in = (const unsigned char*)d_in; a.in_off = (const unsigned long long*)d_in_off; a.in_single = in_single;
    a.n_buf = (uint32_t)n_buf; a.ids = d_ids; a.ids_cap = ids_cap; a.id_off = (unsigned long long*)d_id_off;
    a.n_ids_out = (unsigned long long*)d_n_ids; a.status = d_status; a.sink = sink; a.skip = skip;
    size_t max_blocks = (sink.bm ? (size_t)sink.n_bits : ids_cap) / kBlk + n_buf + 1;
    if (sink.bm && d_in_off) max_blocks = ~(size_t)0 >> 8;       // (streams of a batch may repeat IDs: bounded by the workspace only)
    return t == BFSC_U32 ? launch_decode<32>(a, max_blocks, (cudaStream_t)stream)
                         : launch_decode<64>(a, max_blocks, (cudaStream_t)stream);
}

}  // namespace bfsc

extern "C" bfsc_status bfsc_decompress(const void* d_in, size_t in_bytes, bfsc_dtype t, void* d_ids,
                                       size_t ids_capacity, uint64_t* d_n_ids, void* d_workspace,
                                       size_t workspace_bytes, uint32_t* d_status, void* cuda_stream) {
    if (!d_n_ids) return BFSC_ERR_INVALID_ARG;
    return bfsc::decode_common(d_in, nullptr, in_bytes, 1, t, d_ids, ids_capacity, nullptr, d_n_ids, d_workspace,
                               workspace_bytes, d_status, cuda_stream);
}

extern "C" bfsc_status bfsc_decompress_batch(const void* d_in, const uint64_t* d_in_offsets, size_t n_buf,
                                             bfsc_dtype t, void* d_ids, size_t ids_capacity,
                                             uint64_t* d_id_offsets, void* d_workspace, size_t workspace_bytes,
                                             uint32_t* d_status, void* cuda_stream) {
    if (!d_in_offsets || !d_id_offsets) return BFSC_ERR_INVALID_ARG;
    return bfsc::decode_common(d_in, d_in_offsets, 0, n_buf, t, d_ids, ids_capacity, d_id_offsets, nullptr,
                               d_workspace, workspace_bytes, d_status, cuda_stream);
}

#ifdef BFSC_CHECKED
extern "C" void bfsc_debug_checks_decode(unsigned int* h_failures_and_line) {      // BFSC_CHECK violations of the decode kernels so far
    cudaDeviceSynchronize();
    cudaMemcpyFromSymbol(h_failures_and_line, bfsc::g_bfsc_check, 2 * sizeof(unsigned int));
}
#endif

extern "C" bfsc_status bfsc_decompress_to_bitmap(const void* d_in, size_t in_bytes, bfsc_dtype t, uint64_t id_base,
                                                 uint32_t* d_bitmap, size_t n_bits, uint64_t* d_n_ids,
                                                 void* d_workspace, size_t workspace_bytes, uint32_t* d_status,
                                                 void* cuda_stream) {
    if (!d_n_ids || !d_bitmap || ((uintptr_t)d_bitmap & 15) || n_bits > (1ull << 32)) return BFSC_ERR_INVALID_ARG;
    return bfsc::decode_common(d_in, nullptr, in_bytes, 1, t, nullptr, ~(size_t)0, nullptr, d_n_ids, d_workspace,
                               workspace_bytes, d_status, cuda_stream, bfsc::BitSink{d_bitmap, id_base, n_bits, d_status, nullptr});
}

extern "C" bfsc_status bfsc_decompress_to_frontier(const void* d_in, size_t in_bytes, bfsc_dtype t, uint64_t id_base,
                                                   uint32_t* d_frontier, uint32_t* d_visited, size_t n_bits,
                                                   uint64_t* d_n_ids, void* d_workspace, size_t workspace_bytes,
                                                   uint32_t* d_status, void* cuda_stream) {
    if (!d_n_ids || !d_frontier || !d_visited || d_frontier == d_visited || ((uintptr_t)d_frontier & 15) ||
        ((uintptr_t)d_visited & 15) || n_bits > (1ull << 32))
        return BFSC_ERR_INVALID_ARG;
    return bfsc::decode_common(d_in, nullptr, in_bytes, 1, t, nullptr, ~(size_t)0, nullptr, d_n_ids, d_workspace,
                               workspace_bytes, d_status, cuda_stream, bfsc::BitSink{d_frontier, id_base, n_bits, d_status, d_visited});
}

extern "C" bfsc_status bfsc_decompress_batch_to_frontier(const void* d_in, const uint64_t* d_in_offsets, size_t n_buf,
                                                         bfsc_dtype t, uint64_t id_base, uint32_t* d_frontier,
                                                         uint32_t* d_visited, size_t n_bits, uint64_t* d_n_ids,
                                                         void* d_workspace, size_t workspace_bytes, uint32_t* d_status,
                                                         void* cuda_stream) {
    if (!d_in_offsets || !d_n_ids || !d_frontier || d_frontier == d_visited || ((uintptr_t)d_frontier & 15) ||
        ((uintptr_t)d_visited & 15) || n_bits > (1ull << 32))
        return BFSC_ERR_INVALID_ARG;
    return bfsc::decode_common(d_in, d_in_offsets, 0, n_buf, t, nullptr, ~(size_t)0, nullptr, d_n_ids, d_workspace,
                               workspace_bytes, d_status, cuda_stream, bfsc::BitSink{d_frontier, id_base, n_bits, d_status, d_visited});
}

// ---- FORMAT.md §10: the (visited) bitmap container. begin (parse the header; kind 0: the payload is the bitmap; else the
// scratch bitmap is cleared) -> the decode kernel into the scratch bitmap (skipped for kind 0 / a rejected container) ->
// end (the scratch bitmap, or its complement, becomes the caller's; a rejected container leaves the caller's bitmap as
// it was).
namespace bfsc {
struct VbScratch { unsigned long long count, stream_bytes, n_decoded, n_listed; unsigned int status, kind, skip, pad; };
__global__ void __launch_bounds__(256) k_vb_begin(const unsigned char* __restrict__ in, unsigned long long in_bytes, unsigned long long n_bits,
                                                  uint32_t* __restrict__ wb, uint32_t* __restrict__ bitmap, VbScratch* sc, uint32_t* status) {
    pdl_wait();                                                          // the call before this one is complete (workspace, inputs)
    pdl_launch_dependents();
    const unsigned long long words = (n_bits + 31) / 32, raw_bytes = (4 * words + 15) & ~15ull;
    uint32_t err = 0, kind = 0;
    unsigned long long total = 0, n_listed = 0;
    if (in_bytes < 32) err = BFSC_ERR_CORRUPT;
    else {
        const uint4 h0 = *reinterpret_cast<const uint4*>(in), h1 = *reinterpret_cast<const uint4*>(in + 16);
        kind = (h0.y >> 16) & 0xffu;
        const unsigned long long nb = (unsigned long long)h0.w << 32 | h0.z;
        total = (unsigned long long)h1.y << 32 | h1.x;
        n_listed = (unsigned long long)h1.w << 32 | h1.z;
        if (h0.x != 0x56534642u || (h0.y & 0xffu) != 1u || ((h0.y >> 8) & 0xffu) != 32u || kind > 2u || (h0.y >> 24) != 0u) err = BFSC_ERR_CORRUPT;
        else if (total > in_bytes || (total & 15) || total < 32) err = BFSC_ERR_CORRUPT;
        else if (nb != n_bits) err = BFSC_ERR_DST_TOO_SMALL;
        else if (kind == 0u) {
            if (total != 32 + raw_bytes || n_listed != 0) err = BFSC_ERR_CORRUPT;
            else                                                         // the pad behind bit n_bits - 1 is zero
                for (unsigned long long w = n_bits / 32; w < raw_bytes / 4; w++) {
                    uint32_t x = reinterpret_cast<const uint32_t*>(in + 32)[w];
                    if (w == n_bits / 32 && (n_bits & 31)) x &= ~((1u << (uint32_t)(n_bits & 31)) - 1u);
                    if (x) err = BFSC_ERR_CORRUPT;
                }
        } else {                                                         // the stream inside ends inside the container
            if (total < 64) err = BFSC_ERR_CORRUPT;
            else {
                const uint4 s1 = *reinterpret_cast<const uint4*>(in + 48);
                const unsigned long long inner = (unsigned long long)s1.y << 32 | s1.x;
                if (inner + 32 > total) err = BFSC_ERR_CORRUPT;
            }
        }
    }
    const unsigned long long me = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x, stride = (unsigned long long)gridDim.x * blockDim.x;
    if (me == 0) {
        sc->kind = kind; sc->skip = (err != 0u || kind == 0u) ? 1u : 0u; sc->n_listed = n_listed; sc->status = 0; sc->n_decoded = 0;
        sc->pad = err;
        if (err) set_status(status, err);
    }
    if (err) return;
    if (kind == 0u) { for (unsigned long long w = me; w < words; w += stride) bitmap[w] = reinterpret_cast<const uint32_t*>(in + 32)[w]; }
    else for (unsigned long long w = me; w < words + 4; w += stride) wb[w] = 0u;
}
__global__ void __launch_bounds__(256) k_vb_end(const uint32_t* __restrict__ wb, uint32_t* __restrict__ bitmap, unsigned long long n_bits,
                                                const VbScratch* sc, uint32_t* status) {
    pdl_wait();
    pdl_launch_dependents();
    if (sc->skip) return;                                                // kind 0 (done) or rejected
    if (sc->status != 0u || sc->n_decoded != sc->n_listed) {             // the stream inside: malformed, an ID >= n_bits, or not n_listed IDs
        if (blockIdx.x == 0 && threadIdx.x == 0) set_status(status, sc->status == BFSC_ERR_CUDA ? BFSC_ERR_CUDA : BFSC_ERR_CORRUPT);
        return;
    }
    const bool invert = sc->kind == 2u;
    const unsigned long long words = (n_bits + 31) / 32;
    for (unsigned long long w = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; w < words; w += (unsigned long long)gridDim.x * blockDim.x) {
        uint32_t x = invert ? ~wb[w] : wb[w];
        if (w == words - 1 && (n_bits & 31)) x &= (1u << (uint32_t)(n_bits & 31)) - 1u;
        bitmap[w] = x;
    }
}
}  // namespace bfsc

extern "C" bfsc_status bfsc_decompress_vbitmap(const void* d_in, size_t in_bytes, uint32_t* d_bitmap, size_t n_bits,
                                               void* d_workspace, size_t workspace_bytes, uint32_t* d_status, void* cuda_stream) {
    using namespace bfsc;
    if (!d_in || !d_workspace || (n_bits && !d_bitmap) || (unsigned long long)n_bits > (1ull << 32)) return BFSC_ERR_INVALID_ARG;
    if (((uintptr_t)d_in & 15) || ((uintptr_t)d_workspace & 15) || ((uintptr_t)d_bitmap & 3)) return BFSC_ERR_INVALID_ARG;
    if (workspace_bytes < bfsc_vbitmap_workspace_bytes(n_bits)) return BFSC_ERR_INVALID_ARG;
    cudaStream_t s = (cudaStream_t)cuda_stream;
    DeviceInfo dev;
    if (!current_device(&dev)) return BFSC_ERR_CUDA;
    const size_t words = (n_bits + 31) / 32, wb_bytes = align_up(4 * words + 16, 256);
    VbScratch* sc = reinterpret_cast<VbScratch*>(d_workspace);
    uint32_t* wb = reinterpret_cast<uint32_t*>(static_cast<char*>(d_workspace) + 256);
    void* ws_std = static_cast<char*>(d_workspace) + 256 + wb_bytes;
    int grid = (int)((words + 255) / 256);
    if (grid > dev.sms * 8) grid = dev.sms * 8;
    if (grid < 1) grid = 1;
    BFSC_LAUNCH(launch_dep_v(k_vb_begin, grid, 256, 0, s, static_cast<const unsigned char*>(d_in), (unsigned long long)in_bytes,
                             (unsigned long long)n_bits, wb, d_bitmap, sc, d_status));
    const bfsc_status rc = decode_common(static_cast<const unsigned char*>(d_in) + 32, nullptr, in_bytes >= 32 ? in_bytes - 32 : 0, 1, BFSC_U32,
                                         nullptr, ~(size_t)0, nullptr, reinterpret_cast<uint64_t*>(&sc->n_decoded), ws_std,
                                         workspace_bytes - 256 - wb_bytes, &sc->status, cuda_stream,
                                         BitSink{wb, 0, n_bits, &sc->status, nullptr}, &sc->skip);
    if (rc != BFSC_OK) return rc;
    BFSC_LAUNCH(launch_dep_v(k_vb_end, grid, 256, 0, s, (const uint32_t*)wb, d_bitmap, (unsigned long long)n_bits, (const VbScratch*)sc, d_status));
    return BFSC_OK;
}
