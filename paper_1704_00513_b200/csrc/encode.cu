// encode.cu — bfsc_compress / bfsc_compress_batch (steps E0-E5).
//
// Launches per call, chained with programmatic dependent launch (a dependent kernel starts while its predecessor still
// runs and executes griddepcontrol.wait before it touches what the predecessor writes):
//   one buffer              k_enc_plan -> k_enc_tiles<W, 0> [-> k_enc_streams: no block at all] [-> k_enc_fallback: FORMAT.md §8]
//   small batch             k_enc_small (one cluster; <= 1024 buffers, <= 2048 blocks by the workspace size)
//   batch                   k_enc_planblocks (<= 8192 buffers; else k_enc_plan -> k_enc_blocks) -> k_enc_tiles<W, 1> -> k_enc_streams
//   frontier bitmap         k_bm_count -> k_bm_plan -> k_bm_starts (block starts; sparse bitmaps: the ID list instead) -> k_enc_tiles<W, 2> -> k_bm_finish
//   batch, scattered        as `batch` / `small batch` with k_enc_tiles<W, 3>: every stream to its own destination address (bfsc_compress_batch_scatter)
//   visited bitmap          k_vb_count -> k_vb_select -> the frontier-bitmap chain on the selected copy -> k_vb_finish (FORMAT.md §10)
#include <mutex>

#include "bitmap_stage.cuh"
#include "quad_encode.cuh"
#include "wide_encode.cuh"

namespace bfsc {

struct EncArgs {
    const void* ids;
    const unsigned long long* in_off;   // n_buf+1 element offsets, or nullptr (single buffer of n_single IDs)
    unsigned long long n_single;
    const uint32_t* bitmap;             // bfsc_compress_bitmap (FORMAT.md §9): the IDs are the set bits of bitmap[0 .. n_bits), + id_base;
    unsigned long long n_bits, id_base; //   their number is counted on the device (ws.hdr->n_ids); ids == nullptr then
    unsigned long long* super;          //   bitmap: set bits before every super-chunk of 32 chunks (n_super + 1 entries, behind the standard workspace and `chunk`)
    uint32_t* chunk;                    //   bitmap: set bits of every 1024-bit chunk (32 n_super entries, before `super`)
    unsigned long long n_chunks, n_super;
    void* list;                         //   bitmap, sparse (at most one set bit in 16): the IDs written out by k_bm_starts (behind `super`), staged by the
                                        //   tile kernel like an ID array; denser bitmaps are expanded inside the tile kernel (bm_expand)
    uint32_t fallback;                  // BFSC_CODEC_FLAG_RAW_FALLBACK (FORMAT.md §8), single-buffer calls
    uint32_t n_buf;
    uint32_t codec;                     // encoder rule = mode byte: 1 PFOR-D1 (E2: size argmin), 2 BP128-D1 (b = maxw, no exceptions; FORMAT.md §7)
    uint32_t exclusive;                 // BFSC_CODEC_FLAG_EXCLUSIVE: the CTAs' first two tiles are static (grid CTAs; tickets start at 2 grid)
    uint32_t grid;                      // CTAs of k_enc_tiles
    unsigned long long thr;             // raw threshold in bytes
    unsigned char* out;
    unsigned long long out_cap;
    unsigned long long* out_off;        // n_buf+1 (batch) or nullptr
    unsigned long long* out_total;      // single: *d_out_bytes, or nullptr
    const unsigned long long* dst;      // bfsc_compress_batch_scatter: n_buf device ADDRESSES, stream i is written at dst[i] (out == nullptr,
    unsigned long long dst_cap;         //   out_cap == ~0: `out + offset` below is the address itself); bytes behind every dst[i]
    unsigned long long* out_sizes;      //   n_buf stream sizes (0: the stream did not fit / bad address)
    uint32_t* status;
    WsView ws;
};

__device__ __forceinline__ unsigned long long buf_start(const EncArgs& a, uint32_t i) {
    return a.in_off ? a.in_off[i] : 0ull;
}
__device__ __forceinline__ unsigned long long buf_count(const EncArgs& a, uint32_t i) {
    return a.in_off ? a.in_off[i + 1] - a.in_off[i] : a.n_single;
}
// bitmap source: sparse (at most one set bit in 16 on average: measured on 2^25 bits, us per compress call, listed / expanded in
// the tile kernel: density 1/4 72 / 47, 1/8 38 / 35, 1/16 23 / 29, 1/25 21 / 31) = the IDs are listed by k_bm_starts
__device__ __forceinline__ bool bm_sparse(const EncArgs& a) { return a.ws.hdr->n_ids * 16ull <= a.n_bits; }


constexpr int kEncWorkers = 8;                           // worker warps per CTA
constexpr int kTileR = kEncWorkers * kQuadBlocks;        // 64 blocks per tile
static_assert(kTileR >= kTileBlocks, "workspace sizing assumes tiles of at least kTileBlocks blocks");
constexpr int kPer = (kTileR + 31) / 32;                 // blocks per lane of the scan warp
constexpr int kEncThreads = (kEncWorkers + 2) * 32;      // + the scan warp + the prep warp
constexpr int kEncCtasPerSm = (kEncWorkers >= 16) ? 1 : 2;
constexpr int kSizesThreads = (kEncWorkers + 1) * 32;    // threads on the "sizes posted" barrier: workers + scan warp

// ---- E0: plan. One CTA; per buffer: mode, block count, fixed bytes; exclusive prefixes. ----
template <int W>
__global__ void __launch_bounds__(1024) k_enc_plan(EncArgs a) {
    __shared__ Scan2 sm[33];
    __shared__ int bad;
    __shared__ HintQueue hq;
    constexpr unsigned long long E = W / 8;
    pdl_wait();                                          // the call before this one is complete (workspace, inputs)
    pdl_launch_dependents();
    if (a.in_off == nullptr) {                           // single buffer: no scan needed
        const unsigned long long n = a.n_single;
        const bool raw = n * E < a.thr;
        const unsigned long long nb = raw ? 0ull : (n + kBlk - 1) / kBlk;
        const unsigned long long fixed = raw ? 32ull + ((n * E + 15ull) & ~15ull) : 32ull + ((4ull * (nb + 1) + 15ull) & ~15ull);
        const unsigned long long nt = (nb + kTileR - 1) / kTileR;
        const bool ok = nb <= a.ws.blk_cap && nt <= a.ws.tile_cap;
        if (ok)
            for (unsigned long long q = threadIdx.x; q < nt; q += blockDim.x) a.ws.tile_state[q * kStateStride] = 0;
        if (threadIdx.x == 0) {
            a.ws.blk_first[0] = 0; a.ws.blk_first[1] = nb;
            a.ws.fixed_prefix[0] = 0; a.ws.fixed_prefix[1] = fixed;
            a.ws.stream_start[0] = 0; a.ws.stream_start[1] = 0;
            a.ws.hdr->total_blocks = nb; a.ws.hdr->fixed_total = fixed; a.ws.hdr->ticket = a.exclusive ? 2 * a.grid : 0;
            a.ws.hdr->grand16 = 0; a.ws.hdr->total_out = fixed; a.ws.hdr->ok = ok ? 1u : 0u;
            if (!ok) set_status(a.status, BFSC_ERR_INVALID_ARG);
        }
        return;
    }
    if (threadIdx.x == 0) { bad = 0; hq.n = 0; }
    __syncthreads();
    Scan2 carry{0, 0};
    constexpr int kIpt = 4;                              // buffers per thread and round: 4096 buffers per block scan
    for (uint32_t i0 = 0; i0 < a.n_buf; i0 += blockDim.x * kIpt) {
        Scan2 v[kIpt], sum{0, 0};
#pragma unroll
        for (int u = 0; u < kIpt; u++) {
            const uint32_t i = i0 + threadIdx.x * kIpt + u;
            v[u] = Scan2{0, 0};
            if (i < a.n_buf) {
                if (a.in_off[i + 1] < a.in_off[i]) bad = 1;
                const unsigned long long n = buf_count(a, i);
                const bool raw = n * E < a.thr;                           // FORMAT.md §1 (L1311)
                const unsigned long long nb = raw ? 0ull : (n + kBlk - 1) / kBlk;
                v[u].a = nb;
                v[u].b = raw ? 32ull + ((n * E + 15ull) & ~15ull) : 32ull + ((4ull * (nb + 1) + 15ull) & ~15ull);
            }
            sum.a += v[u].a; sum.b += v[u].b;
        }
        Scan2 tot;
        Scan2 ex = block_scan_excl2(sum, &tot, sm);
        ex.a += carry.a; ex.b += carry.b;
        // The thread's four table entries leave as 16-byte stores (the tables are 16-byte aligned, the thread's
        // first buffer is a multiple of 4): one SM writes all of them, and 8-byte stores at a 32-byte stride cost
        // a sector write each (4096 buffers: 7 us of an 11 us plan).
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
                *reinterpret_cast<ulonglong2*>(a.ws.stream_start + ib + u) = make_ulonglong2(0ull, 0ull);
            }
        } else {
#pragma unroll
            for (int u = 0; u < kIpt; u++)
                if (ib + u < a.n_buf) { a.ws.blk_first[ib + u] = bf[u]; a.ws.fixed_prefix[ib + u] = fp[u]; a.ws.stream_start[ib + u] = 0; }
        }
        carry.a += tot.a; carry.b += tot.b;
        plan_hints_flush(a.ws.tile_state, a.ws.tile_cap, &hq);
    }
    __syncthreads();
    {                                                    // look-back states start invalid
        unsigned long long nt = (carry.a + kTileR - 1) / kTileR;
        if (nt > a.ws.tile_cap) nt = a.ws.tile_cap;
        for (unsigned long long q = threadIdx.x; q < nt; q += blockDim.x) a.ws.tile_state[q * kStateStride] = 0;
    }
    if (threadIdx.x == 0) a.ws.blk_first[a.n_buf] = carry.a;
    if (threadIdx.x == 0) {
        a.ws.fixed_prefix[a.n_buf] = carry.b;
        a.ws.stream_start[a.n_buf] = 0;
        a.ws.hdr->total_blocks = carry.a;
        a.ws.hdr->fixed_total = carry.b;
        a.ws.hdr->ticket = a.exclusive ? 2 * a.grid : 0;
        a.ws.hdr->grand16 = 0;
        a.ws.hdr->total_out = carry.b;
        const bool ok = !bad && carry.a <= a.ws.blk_cap && (carry.a + kTileR - 1) / kTileR <= a.ws.tile_cap;
        a.ws.hdr->ok = ok ? 1u : 0u;
        if (!ok) set_status(a.status, BFSC_ERR_INVALID_ARG);
    }
}

// ---- E0 (batch calls), second part: the block table. One thread per block of the batch: its buffer
// (search from the group hint: one or two cached loads), first ID and valid IDs -> ws.blk_tab, so that
// k_enc_tiles finds a block with one load instead of a chain of dependent ones.
constexpr int kBlkTabThreads = 256;
template <int W>
__global__ void __launch_bounds__(kBlkTabThreads) k_enc_blocks(EncArgs a) {
    pdl_wait();
    pdl_launch_dependents();
    if (a.ws.hdr->ok == 0) return;
    const unsigned long long total = a.ws.hdr->total_blocks;
    EncBlk* tab = reinterpret_cast<EncBlk*>(a.ws.blk_tab);
    for (unsigned long long g = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; g < total;
         g += (unsigned long long)gridDim.x * blockDim.x) {
        const uint32_t i = find_buf_from(a.ws.blk_first, a.n_buf, g, group_hint(a.ws.tile_state, g));
        const unsigned long long k = g - a.ws.blk_first[i], n = buf_count(a, i);
        uint4 e;
        const unsigned long long xoff = buf_start(a, i) + kBlk * k;
        e.x = (uint32_t)xoff; e.y = (uint32_t)(xoff >> 32);
        e.z = (uint32_t)min((unsigned long long)kBlk, n - kBlk * k); e.w = i;
        reinterpret_cast<uint4*>(tab + g)[0] = e;        // (the second half of the entry is unused by encode)
    }
}

// ---- E0 (batch calls of up to kFusedMaxBuf buffers): plan AND block table in ONE launch of many CTAs. Every CTA
// repeats the whole scan over the buffers for itself (n_buf + 1 offsets from L2, one block scan: no inter-CTA
// dependency, no second launch whose start has to wait for the first one's end) and keeps the buffers' first blocks
// in shared memory; it then writes ITS slice of everything: per-buffer tables, look-back states, group hints, and
// the block table (buffer of a block: bisection in shared memory). Replaces k_enc_plan -> k_enc_blocks.
constexpr uint32_t kFusedMaxBuf = 8192;
constexpr int kFusedIpt = 8;                             // buffers per thread (1024 threads)
__device__ __forceinline__ uint32_t bisect_first(const uint32_t* __restrict__ first, uint32_t n_buf, uint32_t g) {
    uint32_t lo = 0, hi = n_buf;                         // the last i in [0, n_buf) with first[i] <= g (first[0] = 0)
    while (hi - lo > 1) {
        const uint32_t mid = (lo + hi) >> 1;
        if (first[mid] <= g) lo = mid; else hi = mid;
    }
    return lo;
}
template <int W>
__global__ void __launch_bounds__(1024) k_enc_planblocks(EncArgs a) {
    __shared__ Scan2 sm[33];
    __shared__ uint32_t s_first[kFusedMaxBuf + 1];
    __shared__ int bad;
    constexpr unsigned long long E = W / 8;
    pdl_wait();                                          // the call before this one is complete (workspace, inputs)
    pdl_launch_dependents();
    if (threadIdx.x == 0) bad = 0;
    __syncthreads();
    const uint32_t ib = threadIdx.x * kFusedIpt;
    Scan2 v[kFusedIpt], sum{0, 0};
#pragma unroll
    for (int u = 0; u < kFusedIpt; u++) {
        const uint32_t i = ib + u;
        v[u] = Scan2{0, 0};
        if (i < a.n_buf) {
            const unsigned long long o0 = a.in_off[i], o1 = a.in_off[i + 1];
            if (o1 < o0) bad = 1;
            const unsigned long long n = o1 - o0;
            const bool raw = n * E < a.thr;                               // FORMAT.md §1 (L1311)
            const unsigned long long nb = raw ? 0ull : (n + kBlk - 1) / kBlk;
            v[u].a = nb;
            v[u].b = raw ? 32ull + ((n * E + 15ull) & ~15ull) : 32ull + ((4ull * (nb + 1) + 15ull) & ~15ull);
        }
        sum.a += v[u].a; sum.b += v[u].b;
    }
    Scan2 tot;
    Scan2 ex = block_scan_excl2(sum, &tot, sm);
    const bool mine = threadIdx.x % gridDim.x == blockIdx.x;              // table entries of this thread's buffers: this CTA's
#pragma unroll
    for (int u = 0; u < kFusedIpt; u++) {
        const uint32_t i = ib + u;
        if (i < a.n_buf) {
            s_first[i] = (uint32_t)ex.a;
            if (mine) { a.ws.blk_first[i] = ex.a; a.ws.fixed_prefix[i] = ex.b; a.ws.stream_start[i] = 0; }
        }
        ex.a += v[u].a; ex.b += v[u].b;
    }
    if (threadIdx.x == 0) s_first[a.n_buf] = (uint32_t)tot.a;
    __syncthreads();
    const unsigned long long total = tot.a, nt = (total + kTileR - 1) / kTileR;
    const bool ok = !bad && total <= a.ws.blk_cap && nt <= a.ws.tile_cap && total < (1ull << 32);
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        a.ws.blk_first[a.n_buf] = total; a.ws.fixed_prefix[a.n_buf] = tot.b; a.ws.stream_start[a.n_buf] = 0;
        a.ws.hdr->total_blocks = total; a.ws.hdr->fixed_total = tot.b; a.ws.hdr->ticket = a.exclusive ? 2 * a.grid : 0;
        a.ws.hdr->grand16 = 0; a.ws.hdr->total_out = tot.b; a.ws.hdr->ok = ok ? 1u : 0u;
        if (!ok) set_status(a.status, BFSC_ERR_INVALID_ARG);
    }
    if (!ok) return;
    const unsigned long long stride = (unsigned long long)gridDim.x * blockDim.x;
    for (unsigned long long t = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; t < nt; t += stride) {
        a.ws.tile_state[t * kStateStride] = 0;                            // look-back states start invalid
        a.ws.tile_state[t * kStateStride + 1] = bisect_first(s_first, a.n_buf, (uint32_t)(t * kTileR));   // group hint
    }
    EncBlk* tab = reinterpret_cast<EncBlk*>(a.ws.blk_tab);
    for (unsigned long long g = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; g < total; g += stride) {
        const uint32_t i = bisect_first(s_first, a.n_buf, (uint32_t)g);
        const unsigned long long k = g - s_first[i], o0 = a.in_off[i], n = a.in_off[i + 1] - o0;
        const unsigned long long xoff = o0 + kBlk * k;
        uint4 e;
        e.x = (uint32_t)xoff; e.y = (uint32_t)(xoff >> 32);
        e.z = (uint32_t)min((unsigned long long)kBlk, n - kBlk * k); e.w = i;
        reinterpret_cast<uint4*>(tab + g)[0] = e;        // (the second half of the entry is unused by encode)
    }
}

// ---- E1-E4 fused: one pass over HBM ------------------------------------------------------
// CTA = 8 worker warps + 1 scan warp; tile = 64 consecutive blocks (32 KB of u32 IDs), pulled by
// ticket. Worker warps handle 8 blocks each, four lanes per block (quad_encode.cuh):
//   E1+E2  load (128-bit, streaming), deltas, canonical b  -> s_key, arrive on barrier 1
//   E4     stage deltas -> column owners mask + pack the payload, exceptions, header into the
//          warp's image area (shared memory) — overlapped with the scan warp's E3
//   sync on barrier 2, copy the image to its final offset with 128-bit stores.
// Scan warp (E3): while the workers run E1/E2 it draws the next ticket and prepares that tile's
// bookkeeping; after barrier 1: intra-tile exclusive scan of the 64 sizes, aggregate published,
// decoupled look-back over the tiles in flight (= device-wide exclusive scan of block sizes),
// final byte offset of every block -> s_at, directory entries, stream starts, and (single-buffer
// calls) the stream header; barrier 2.
constexpr unsigned long long kFlagAgg = 1ull << 62, kFlagPre = 2ull << 62, kValMask = (1ull << 62) - 1;
constexpr unsigned long long kNoTile = ~0ull, kSkip = ~0ull;
constexpr uint32_t kLateBit = 1u << 31;                  // in a stored key: the block is assembled by late_emit, not in an image buffer
constexpr uint32_t kDoneBit = 1u << 30;                  // in a stored key: the block is in the output already (packed straight from the registers)

__device__ __forceinline__ unsigned long long ld_volatile_u64(const unsigned long long* p) {
    unsigned long long v;
    asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");   // gpu scope: the writers are CTAs of this grid
    return v;
}
__device__ __forceinline__ void st_volatile_u64(unsigned long long* p, unsigned long long v) {
    asm volatile("st.relaxed.gpu.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}
// mbarrier (shared memory, CTA scope): one-directional "posted" signals between warps of a CTA
__device__ __forceinline__ void mbar_init(unsigned long long* b, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"((uint32_t)__cvta_generic_to_shared(b)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(unsigned long long* b) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"((uint32_t)__cvta_generic_to_shared(b)) : "memory");
}
__device__ __forceinline__ bool mbar_test(uint32_t addr, uint32_t parity) {
    uint32_t ok;
    asm volatile("{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n selp.u32 %0, 1, 0, p;\n}"
                 : "=r"(ok) : "r"(addr), "r"(parity) : "memory");
    return ok != 0;
}
// Until the phase of that parity has completed. Whole warp calls. A warp that has to wait sleeps between
// polls: a spinning warp would take issue slots from the warps it waits for.
__device__ __forceinline__ void mbar_wait(unsigned long long* b, uint32_t parity) {
    const uint32_t addr = (uint32_t)__cvta_generic_to_shared(b);
    while (!mbar_test(addr, parity)) __nanosleep(64);
}
// Bulk (TMA) store shared -> global, issued by one lane: 16-byte aligned addresses, size a multiple of 16.
__device__ __forceinline__ void bulk_store(void* gdst, const void* ssrc, uint32_t bytes) {
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(gdst),
                 "r"((uint32_t)__cvta_generic_to_shared(ssrc)), "r"(bytes) : "memory");
    asm volatile("cp.async.bulk.commit_group;" ::: "memory");
}
__device__ __forceinline__ void bulk_wait_read() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }   // sources may be overwritten
__device__ __forceinline__ void bulk_wait_all() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }
__device__ __forceinline__ void fence_proxy_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void prefetch_l2_bulk(const void* gsrc, uint32_t bytes) {   // 16-byte aligned, a multiple of 16
    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(gsrc), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bar_arrive(int id, int n) { asm volatile("bar.arrive %0, %1;" ::"r"(id), "r"(n) : "memory"); }
__device__ __forceinline__ void bar_sync(int id, int n) { asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(n) : "memory"); }

// Decoupled look-back (one warp): the exclusive prefix of tile t > 0 = aggregates of t-1, t-2, ... down to the
// nearest tile whose inclusive prefix is known. Every lane sums its own entries, a single warp reduction ends it.
constexpr int kLookChunks = 1;                       // rounds of 32 predecessor states (the measured optimum, see lookback)
constexpr unsigned kLookSleepNs = 32;                // back-off between polls of a look-back that has to wait
// One round of the look-back: the states of the 32 * N predecessors below idx0 (lane i: idx0 - i, - 32, ...) are
// requested at once, then examined 32 at a time with two ballots; an entry that is not posted yet is polled alone.
template <int N>
__device__ __forceinline__ bool lookback_round(const unsigned long long* __restrict__ state, long long idx, int lane,
                                               unsigned long long& acc) {
    unsigned long long s[N];
    bool done = false;
#pragma unroll
    for (int r = 0; r < N; r++)
        s[r] = (idx - 32 * r >= 0) ? ld_volatile_u64(&state[(idx - 32 * r) * kStateStride]) : kFlagPre;
#pragma unroll
    for (int r = 0; r < N; r++) {
        if (!done) {
            unsigned long long v = s[r];
            while (true) {
                const uint32_t hit = __ballot_sync(kFull, (v >> 62) == 2);
                const uint32_t rdy = __ballot_sync(kFull, (v >> 62) != 0);
                const int stop = hit ? __ffs(hit) - 1 : 31;
                const uint32_t need = 0xffffffffu >> (31 - stop);
                if ((rdy & need) == need) {
                    if (lane <= stop) acc += v & kValMask;
                    done = hit != 0;
                    break;
                }
                __nanosleep(kLookSleepNs);
                if ((v >> 62) == 0) v = ld_volatile_u64(&state[(idx - 32 * r) * kStateStride]);
            }
        }
    }
    return done;
}

// Exclusive prefix (16-byte units) of tile t > 0: rounds of kLookChunks x 32 predecessor states. One chunk per
// round is the measured optimum (swept 1..24, also with a larger window after the first round, and 4..32
// lanes in the first round): the nearest tile with a known inclusive prefix is usually a few tiles back, and every
// speculative load of a state that other SMs are about to write slows the call (8 chunks: + 1.3 us per call).
__device__ __forceinline__ unsigned long long lookback(const unsigned long long* __restrict__ state,
                                                       unsigned long long t, int lane) {
    unsigned long long acc = 0;
    long long idx = (long long)t - 1 - lane;
    bool done = false;
    while (!done) {
        done = lookback_round<kLookChunks>(state, idx, lane, acc);
        idx -= 32 * kLookChunks;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(kFull, acc, o);
    return acc;
}

// Image buffer of a warp: room for 8 block images of at most kCap bytes, back to back. u32: 544 B — EVERY u32
// block fits (b = 32 costs 528 B and the argmin never exceeds it): nearly incompressible u32 input stays on the
// fast path (with 320-byte slots a stream of 22-bit gaps took 141 us instead of 37). u64: 288 B (b = 17), so that
// two CTAs of the batch instantiation (1 KB blocks staged, 10 KB of bookkeeping) still fit one SM; larger u64
// blocks (gaps over 2^17 between sorted 64-bit IDs) take the slow path.
// kSrc: where the IDs come from — 0: one ID array, 1: a batch of ID arrays, 2: a frontier bitmap (FORMAT.md §9), 3: a batch
// whose streams go to one destination address each (bfsc_compress_batch_scatter) instead of back to back. A bitmap
// has no ID array for the slow path to re-read, so its image slots hold every block (544 B) for both widths (deltas of a
// bitmap of < 2^32 bits fit 32 bits), and each worker warp gets a landing area for the bitmap words of its 8 blocks.
template <int W, int kSrc = 0> struct ImgCfg {
    static constexpr int kSlotChunks = (W == 32 || kSrc == 2) ? 34 : 18;   // 16-byte chunks per block
    static constexpr int kCap = kSlotChunks * 16;                          // bytes of a block image the fast path can hold
    static constexpr int kBufChunks = kQuadBlocks * kSlotChunks;
};

constexpr int kDefer = 1;                                     // a tile's images leave kDefer tiles after they were packed
constexpr int kNB = kDefer + 1;                               // image buffers / size and offset tables per CTA
constexpr int kLandChunks = 32;                               // bitmap words of a warp batch staged by cp.async: 512 B = 4096 bits (denser than 1 ID in 4 bits on average; sparser batches are read from global memory)

template <int W, int kSrc = 0> struct EncSmem {
    static constexpr int kStageChunks = RawCfg<W>::kAreaChunks;              // per worker warp: staged raw IDs
    static constexpr int kWarpChunks = kStageChunks + kNB * ImgCfg<W, kSrc>::kBufChunks + (kSrc == 2 ? kLandChunks : 0);   // + the image buffers (+ landing area)
    static constexpr size_t kBytes = (size_t)kEncWorkers * kWarpChunks * 16;
};

enum { kBarSizes = 1 };                                       // named barriers kBarSizes + tile count mod kNB
constexpr int kRing = 8;                                      // ring of tile bookkeeping slots (workers may be two tiles apart)

// k_enc_tiles: CTA = 8 worker warps + 1 scan warp; a CTA's k-th tile is "tile k" below.
//   workers, iteration k:  E1/E2 of tile k -> sizes in s_key[k % kNB], the last warp publishes the tile's
//       aggregate; exceptions; next tile's raw IDs prefetched (cp.async) into the staging slots; payload
//       packed into image buffer k % kNB; then the offsets of tile k - kDefer are awaited and its images
//       copied out. Worker warp 0 also draws the tickets and prepares the bookkeeping, two tiles ahead.
//   scan warp, tile k: sizes -> intra-tile scan -> decoupled look-back (device-wide exclusive scan of
//       the block sizes) -> final offsets in s_at[k % kNB], directory entries, stream starts, header.
//       It may lag up to kDefer tiles behind the workers: a look-back that waits for a slow
//       predecessor CTA does not stall this CTA's workers.
// Tiles: every one comes from the ticket counter (prep warp), each drawn at the same point of the pipeline: a lower
// tile number means "sizes posted earlier" — and is held by a running CTA, whatever else occupies the device.
template <int W, int kSrc>
__global__ void __launch_bounds__(kEncThreads, kEncCtasPerSm) k_enc_tiles(EncArgs a) {
    using T = typename IdT<W>::T;
    constexpr bool kBatch = kSrc == 1 || kSrc == 3, kBits = kSrc == 2, kScatter = kSrc == 3;
    using Img = ImgCfg<W, kSrc>;
    using Smem = EncSmem<W, kSrc>;
    extern __shared__ __align__(16) uint4 dyn_smem[];    // per worker warp: staging area | kNB image buffers
    __shared__ uint32_t s_key[kNB][kTileR];              // workers: size<<14 | (64-b)<<7 | n_exc, 0 = no block
    __shared__ unsigned long long s_at[kNB][kTileR];     // scan warp: final byte offset of the block, or kSkip
    __shared__ uint32_t s_off16[kTileR];                 // exclusive scan of the sizes inside the tile (16-B units)
    // Ring of tile bookkeeping (batch calls only: a single buffer's blocks follow from the tile number).
    constexpr int kBk = kBatch ? kTileR : 1;
    __shared__ int s_m[kRing][kBk];                          // valid IDs of each block (0 = none)
    __shared__ unsigned long long s_xoff[kRing][kBk];        // element offset of the block's first ID
    __shared__ uint32_t s_buf[kRing][kBk];                   // buffer of each block
    __shared__ unsigned long long s_tile[kRing];             // tile of each ring slot, kNoTile = done
    __shared__ unsigned long long mb_post[kRing];        // warp 0 -> workers: the ring slot's tile is posted (use u of a slot: parity u & 1)
    __shared__ unsigned long long mb_off[kNB];           // scan warp -> workers: the offsets in s_at[kp] are posted
    __shared__ volatile unsigned int s_sized;            // scan warp: tiles of this CTA whose sizes have arrived (the prep warp follows it)
    __shared__ unsigned int s_agg[4];                    // arrivals << 24 | sum of the worker warps' sizes (16-B units)

    // Roles by hardware warp: 0 = prep warp, 1..kEncWorkers = workers, kEncWorkers + 1 = scan warp. The schedulers
    // favour the highest warp number among eligible warps: the scan warp (every later tile waits for its prefix)
    // goes first, the prep warp (runs ahead, polls) last. `warp` below is the ROLE: workers 0..kEncWorkers-1,
    // scan warp kEncWorkers, prep warp kEncWorkers + 1.
    const int hw_warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int warp = hw_warp == 0 ? kEncWorkers + 1 : hw_warp - 1;
    constexpr bool batch = kBatch;
    const T* ids = reinterpret_cast<const T*>(a.ids);
    pdl_launch_dependents();                             // the next call's first kernel may be set up; it waits for this grid
    if constexpr (kSrc == 0) {
        // Single-buffer calls: the plan kernel (ticket counter, zeroed look-back states) is still running.
        if (a.exclusive) {
            // static first tile (tile blockIdx.x): its loads go out before anything else in the kernel
            if (warp < kEncWorkers) {
                const unsigned long long g = (unsigned long long)blockIdx.x * kTileR + warp * kQuadBlocks + (lane >> 2);
                const unsigned long long nb0 = (a.n_single + kBlk - 1) / kBlk;
                if (g < nb0)
                    quad_prefetch<W>(dyn_smem + warp * Smem::kWarpChunks + raw_slot_chunk<W>(lane >> 2), ids + kBlk * g,
                                     (int)min((unsigned long long)kBlk, a.n_single - kBlk * g));
            }
        } else if (warp < kEncWorkers && lane == 0) {
            // Meanwhile pull the tile this CTA will most likely draw first (tickets go out in launch order) into L2.
            const unsigned long long g = (unsigned long long)blockIdx.x * kTileR + warp * kQuadBlocks;
            const unsigned long long nb0 = (a.n_single + kBlk - 1) / kBlk;
            if (g < nb0) {
                const unsigned long long n_el = min((unsigned long long)(kQuadBlocks * kBlk), a.n_single - kBlk * g);
                const uint32_t bytes = (uint32_t)(n_el * sizeof(T)) & ~15u;
                if (bytes) prefetch_l2_bulk(ids + kBlk * g, bytes);
            }
        }
    }
    if (threadIdx.x < 4) s_agg[threadIdx.x] = 0;
    if (threadIdx.x == 4) s_sized = 0;
    if (threadIdx.x < kRing) mbar_init(&mb_post[threadIdx.x], 1);
    if (threadIdx.x >= 32 && threadIdx.x < 32 + kNB) mbar_init(&mb_off[threadIdx.x - 32], 1);
    __syncthreads();

    // n_ids: IDs of the one stream of a single-buffer call — an argument, or (bitmap) counted by the kernels before
    unsigned long long n_ids = a.n_single;
    if constexpr (kBits) {
        pdl_wait();
        n_ids = a.ws.hdr->ok != 0 ? a.ws.hdr->n_ids : 0ull;
    }
    unsigned long long nb_single = (n_ids + kBlk - 1) / kBlk;
    if constexpr (kBits) nb_single = a.ws.hdr->ok != 0 ? a.ws.hdr->total_blocks : 0ull;    // (0: RAW by the threshold, k_bm_finish)
    unsigned long long total = nb_single;
    if (batch) {
        pdl_wait();
        total = a.ws.hdr->ok != 0 ? a.ws.hdr->total_blocks : 0ull;
    }
    const unsigned long long n_tiles = (total + kTileR - 1) / kTileR;
    // bitmap source: ring of the tiles' block starts (bit index of each block's first ID; entry 64 = end of the tile's
    // last block), copied from ws.blk_tab (k_bm_starts) by the prep warp
    constexpr int kSt = kBits ? kTileR + 1 : 1;
    __shared__ uint32_t s_start[kRing][kSt];
    const uint32_t* starts = reinterpret_cast<const uint32_t*>(a.ws.blk_tab);

    auto prep = [&](unsigned long long t, int p) {       // bookkeeping of tile t into ring slot p (one warp)
        if (lane == 0) s_tile[p] = t;
        if (t == kNoTile) return;
        if constexpr (kBatch) {
          for (int jj = lane; jj < kTileR; jj += 32) {
            const unsigned long long g = t * kTileR + jj;
            int m = 0; uint32_t i = 0; unsigned long long xoff = 0;
            if (g < total) {                             // ws.blk_tab, written by k_enc_blocks
                const uint4 e = __ldcg(reinterpret_cast<const uint4*>(reinterpret_cast<const EncBlk*>(a.ws.blk_tab) + g));
                xoff = (unsigned long long)e.y << 32 | e.x; m = (int)e.z; i = e.w;
            }
            s_m[p][jj] = m; s_xoff[p][jj] = xoff; s_buf[p][jj] = i;
          }
        }
        if constexpr (kBits) {
            for (int jj = lane; jj <= kTileR; jj += 32) {
                const unsigned long long g = min(t * kTileR + jj, total);        // starts[total] = n_bits
                s_start[p][jj] = __ldcg(starts + g);
            }
        }
    };
    // valid IDs / element offset of block jj of the tile in ring slot p (the tile is posted and not kNoTile)
    auto blk_m = [&](int p, int jj) -> int {
        if constexpr (kBatch) return s_m[p][jj];
        else {
            const unsigned long long g = s_tile[p] * kTileR + jj;
            return g < nb_single ? (int)min((unsigned long long)kBlk, n_ids - kBlk * g) : 0;
        }
    };
    auto blk_xoff = [&](int p, int jj) -> unsigned long long {
        if constexpr (kBatch) return s_xoff[p][jj];
        else return kBlk * (s_tile[p] * kTileR + jj);
    };

    if (warp == kEncWorkers) {
        // =============================== scan warp ===============================
        const unsigned long long f1_single = 32ull + ((4ull * (nb_single + 1) + 15ull) & ~15ull);
        if (!batch) pdl_wait();                          // the plan kernel's writes are visible from here on
        int kp = 0;                                      // k % kNB
        for (int k = 0;; k++) {
            mbar_wait(&mb_post[k & (kRing - 1)], (k / kRing) & 1);   // the prep warp has posted the CTA's tile k
            const unsigned long long t = s_tile[k & (kRing - 1)];
            if (t == kNoTile) break;
            // batch calls: the per-buffer constants of this lane's blocks (and the start of a stream that began in an
            // earlier tile, if it is published already) are requested BEFORE the sizes are waited for: the tile was
            // posted two tiles ahead, so their latency hides behind the workers' E1/E2
            const unsigned long long g0 = t * kTileR;
            unsigned long long bf_first[kPer], bf_f0[kPer], bf_f1[kPer], bf_S[kPer], bf_dst[kPer];
            uint32_t bf_i[kPer];
            if constexpr (kBatch) {
#pragma unroll
                for (int h = 0; h < kPer; h++) {
                    const int jj = kPer * lane + h;
                    bf_i[h] = 0; bf_first[h] = 0; bf_f0[h] = 0; bf_f1[h] = 0; bf_S[h] = 0; bf_dst[h] = 0;
                    if (jj < kTileR && g0 + jj < total) {
                        const uint32_t i = s_buf[k & (kRing - 1)][jj];
                        bf_i[h] = i; bf_first[h] = a.ws.blk_first[i]; bf_f0[h] = a.ws.fixed_prefix[i]; bf_f1[h] = a.ws.fixed_prefix[i + 1];
                        if (i > 0) bf_S[h] = ld_volatile_u64(&a.ws.stream_start[i]);     // (0: not known yet, or the stream begins in this tile)
                        if constexpr (kScatter) bf_dst[h] = a.dst[i];
                    }
                }
            }
            bar_sync(kBarSizes + kp, kSizesThreads);
            if (lane == 0) s_sized = (unsigned int)k + 1u;      // the workers' sizes of tile t are in s_key[kp]

            // E3: intra-tile scan (kPer consecutive blocks per lane)
            uint32_t kk[kPer], offs[kPer], inc = 0;
#pragma unroll
            for (int h = 0; h < kPer; h++) {
                const int jj = kPer * lane + h;
                kk[h] = jj < kTileR ? s_key[kp][jj] : 0u;
                offs[h] = inc;
                inc += kk[h] >> 18;
            }
            const uint32_t own = inc;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const uint32_t y = __shfl_up_sync(kFull, inc, o);
                if (lane >= o) inc += y;
            }
            const unsigned long long agg = __shfl_sync(kFull, inc, 31);
#pragma unroll
            for (int h = 0; h < kPer; h++) {
                offs[h] += inc - own;
                if (kPer * lane + h < kTileR) s_off16[kPer * lane + h] = offs[h];
            }
            const unsigned long long excl = t > 0 ? lookback(a.ws.tile_state, t, lane) : 0ull;
            if (lane == 0) {
                st_volatile_u64(&a.ws.tile_state[t * kStateStride], kFlagPre | (excl + agg));
                if (t == n_tiles - 1) {
                    a.ws.hdr->grand16 = excl + agg;
                    a.ws.hdr->total_out = a.ws.hdr->fixed_total + 16ull * (excl + agg);
                }
            }
            __syncwarp();

            // Stream starts of the streams that BEGIN in this tile go out first, before any lane below polls for
            // the start of a stream that began in an earlier tile: a publish never waits behind a poll.
            if constexpr (kBatch) {
#pragma unroll
                for (int h = 0; h < kPer; h++) {
                    const int jj = kPer * lane + h;
                    if (jj < kTileR && g0 + jj < total && bf_first[h] == g0 + jj)
                        st_volatile_u64(&a.ws.stream_start[bf_i[h]], bf_f0[h] + 16ull * (excl + offs[h]) + 1);
                }
            }
            // Final offsets first: they need the look-back's result and the plan's tables only, and the workers wait
            // for nothing else. The directory entries follow AFTER the offsets are posted: a batch call's entry also
            // needs the start of its stream, which a stream that spans in from an earlier tile gets from that tile's
            // scan warp (a poll) — that wait is now off the workers' path.
            // Scatter calls: a block's place is its offset INSIDE its stream, behind the stream's own destination — so the
            // start of the stream (in the back-to-back layout the scan runs over) is needed before the offsets can be posted.
            unsigned long long at_h[kPer];
#pragma unroll
            for (int h = 0; h < kPer; h++) {
                const int jj = kPer * lane + h;
                at_h[h] = kSkip;
                if (jj >= kTileR) continue;
                if (g0 + jj < total) {
                    unsigned long long f1 = f1_single;
                    if constexpr (kBatch) f1 = bf_f1[h];
                    const unsigned long long at = f1 + 16ull * (excl + offs[h]);
                    if constexpr (kScatter) {
                        unsigned long long S = 0;
                        if (bf_first[h] >= g0) S = bf_f0[h] + 16ull * (excl + s_off16[bf_first[h] - g0]);
                        else if (bf_i[h] > 0) {
                            S = bf_S[h];
                            while (S == 0) S = ld_volatile_u64(&a.ws.stream_start[bf_i[h]]);
                            S -= 1;
                        }
                        const unsigned long long rel = at - S;
                        if (bf_dst[h] == 0 || (bf_dst[h] & 15)) set_status(a.status, BFSC_ERR_INVALID_ARG);
                        else if (rel + (kk[h] >> 14) <= a.dst_cap) at_h[h] = bf_dst[h] + rel;
                        else set_status(a.status, BFSC_ERR_DST_TOO_SMALL);
                    } else {
                        if (at + (kk[h] >> 14) <= a.out_cap) at_h[h] = at;
                        else set_status(a.status, BFSC_ERR_DST_TOO_SMALL);
                    }
                }
                s_at[kp][jj] = at_h[h];
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(&mb_off[kp]);     // offsets of tile k are posted
            // directory entries, stream header of a single-buffer call
#pragma unroll
            for (int h = 0; h < kPer; h++) {
                const int jj = kPer * lane + h;
                if (jj >= kTileR) continue;
                const unsigned long long g = g0 + jj;
                const uint32_t key = kk[h];
                const unsigned long long at = at_h[h];
                if (g < total) {
                    const uint32_t off = offs[h], bytes = key >> 14;
                    unsigned long long first = 0, f0 = 0, f1 = f1_single, S = 0;
                    uint32_t i = 0;
                    if constexpr (kBatch) {
                        i = bf_i[h]; first = bf_first[h]; f0 = bf_f0[h]; f1 = bf_f1[h];
                        if constexpr (kScatter) S = bf_dst[h];           // (`at` is an address here: at - S = the offset in the stream)
                        else if (at != kSkip) {
                            if (first >= g0) S = f0 + 16ull * (excl + s_off16[first - g0]);
                            else if (i > 0) {            // published by the tile that owns the stream's first block
                                S = bf_S[h];
                                while (S == 0) S = ld_volatile_u64(&a.ws.stream_start[i]);
                                S -= 1;
                            }
                        }
                    }
                    BFSC_CHECK(at == kSkip || (at >= S && (kScatter ? 32 + 4 * (g - first) + 4 <= a.dst_cap : S + 32 + 4 * (g - first) + 4 <= a.out_cap)));
                    if (at != kSkip) reinterpret_cast<uint32_t*>(a.out + S + 32)[g - first] = (uint32_t)((at - S) >> 4);
                    if (!batch && g == total - 1) {      // single buffer: stream header, dir[nb], zero pad
                        const unsigned long long tot = f1 + 16ull * (excl + off) + bytes;
                        if (at != kSkip) {
                            uint4 h0, h1;
                            h0.x = 0x43534642u;                                   // "BFSC"
                            h0.y = 1u | ((uint32_t)W << 8) | (a.codec << 16);     // mode = the encoder rule
                            h0.z = (uint32_t)n_ids; h0.w = (uint32_t)(n_ids >> 32);
                            h1.x = (uint32_t)tot; h1.y = (uint32_t)(tot >> 32);
                            h1.z = (uint32_t)nb_single; h1.w = 0;
                            reinterpret_cast<uint4*>(a.out)[0] = h0;
                            reinterpret_cast<uint4*>(a.out)[1] = h1;
                            uint32_t* dir = reinterpret_cast<uint32_t*>(a.out + 32);
                            dir[nb_single] = (uint32_t)(tot >> 4);
                            for (unsigned long long x = nb_single + 1; x < ((nb_single + 1 + 3) & ~3ull); x++) dir[x] = 0;
                        }
                        if (a.out_total) *a.out_total = at != kSkip ? tot : 0ull;
                    }
                }
            }
            kp = kp == kNB - 1 ? 0 : kp + 1;
        }
        return;
    }

    if (warp == kEncWorkers + 1) {
        // =============================== prep warp ===============================
        // Runs ahead of the workers: draws the ticket of the CTA's tile p, prepares its bookkeeping (batch calls:
        // buffer, first ID, valid IDs of every block — a chain of dependent global loads nobody else has to wait
        // for) and posts it. EVERY tile comes from the ticket counter, in order: whatever a CTA waits for (look-back)
        // belongs to a tile with a lower ticket, which a RUNNING CTA holds — no co-residency assumption (two
        // compress grids, or a compress grid next to any other kernel, cannot deadlock). The CTA's second ticket is
        // drawn a moment after its first, when every CTA of the wave has its first (a CTA holding two neighbouring
        // tiles would publish the second one a tile period late, and the tiles above wait for it); from then on
        // the ticket of tile p is drawn when the sizes of tile p - 2 have arrived: every CTA draws at the same
        // point of its pipeline, so a lower tile number means "sizes posted earlier" and look-backs rarely wait;
        // and no worker can still read the ring slot (kRing = 8) that is rewritten.
        // BFSC_CODEC_FLAG_EXCLUSIVE (the caller vouches that every CTA of the grid becomes resident): the first two
        // tiles are blockIdx.x and blockIdx.x + gridDim.x and need neither the plan kernel nor an atomic.
        auto draw = [&]() -> unsigned long long {
            unsigned int ticket = 0;
            if (lane == 0) ticket = atomicAdd(&a.ws.hdr->ticket, 1u);
            ticket = __shfl_sync(kFull, ticket, 0);
            return ticket < n_tiles ? (unsigned long long)ticket : kNoTile;
        };
        if (a.exclusive) {
            const unsigned long long t0 = blockIdx.x, t1 = (unsigned long long)blockIdx.x + gridDim.x;
            prep(t0 < n_tiles ? t0 : kNoTile, 0);
            prep(t0 < n_tiles && t1 < n_tiles ? t1 : kNoTile, 1);
            __syncwarp();
            if (lane == 0) { mbar_arrive(&mb_post[0]); mbar_arrive(&mb_post[1]); }
            if (!batch) pdl_wait();                      // the ticket counter is set by the plan kernel
        } else {
            if (!batch) pdl_wait();                      // the ticket counter is set by the plan kernel
            const unsigned long long t0 = draw();
            prep(t0, 0);
            __syncwarp();
            if (lane == 0) mbar_arrive(&mb_post[0]);
            __nanosleep(1000);
            const unsigned long long t1 = t0 != kNoTile ? draw() : kNoTile;
            prep(t1, 1);
            __syncwarp();
            if (lane == 0) mbar_arrive(&mb_post[1]);
        }
        bool more = s_tile[1] != kNoTile;
        for (int pt = 2; more; pt++) {
            while ((int)s_sized + 1 < pt) __nanosleep(100);    // (measured: 400 ns between polls +0.2 us per call, 1500 ns +1.1 us: a late ticket is a late tile)
            const unsigned long long t = draw();
            more = t != kNoTile;
            prep(t, pt & (kRing - 1));
            __syncwarp();
            if (lane == 0) mbar_arrive(&mb_post[pt & (kRing - 1)]);
        }
        return;
    }

    // =============================== worker warps ===============================
    const int q = lane >> 2, l = lane & 3;
    uint4* area = dyn_smem + warp * Smem::kWarpChunks;
    uint4* slot = area + raw_slot_chunk<W>(q);                           // staging: the quad's raw IDs
    unsigned char* ibuf = reinterpret_cast<unsigned char*>(area + Smem::kStageChunks);   // the warp's kNB image buffers
    const int j = warp * kQuadBlocks + q;
    mbar_wait(&mb_post[0], 0);                                           // the CTA's first tile is posted (by the prep warp)
    bool have = s_tile[0] != kNoTile;
    uint4* land = area + Smem::kStageChunks + kNB * Img::kBufChunks;      // bitmap source: the words of the warp's 8 blocks
    bool listed = false;                                                 // bitmap source, sparse: the IDs come from k_bm_starts' list
    const T* list = reinterpret_cast<const T*>(a.list);
    if constexpr (kBits) {
        static_assert(!kBits || Img::kCap >= 16 + 16 * 32 + 16, "a bitmap has no ID array for the slow path: every block must fit its image slot");
        listed = bm_sparse(a);
        if (have) {
            if (listed) quad_prefetch<W>(slot, list + blk_xoff(0, j), blk_m(0, j));
            else bm_prefetch<kLandChunks>(land, a.bitmap, s_start[0], warp, lane);
        }
    } else {
        if (have && (kBatch || !a.exclusive)) quad_prefetch<W>(slot, ids + blk_xoff(0, j), blk_m(0, j));   // (exclusive single-buffer calls: see the top)
    }
    static_assert(kDefer == 1 || kDefer == 2, "hist selection below");
    uint32_t key_hist[kDefer] = {}, woff_hist[kDefer] = {};              // keys and image places of the tiles that wait in shared memory
    int kp = 0;                                                          // k % kNB
    int n_wait = 0, ke = 0;                                              // tiles packed but not copied out yet; next one to copy out
    for (int k = 0;; k++) {
        uint32_t key = 0, woff = 0;
        bool have_next = false;
        if (have) {
            const int m = blk_m(k & (kRing - 1), j);
            const T* raw = reinterpret_cast<const T*>(slot);
            if constexpr (!kBits) raw += (reinterpret_cast<uintptr_t>(ids + blk_xoff(k & (kRing - 1), j)) & 15) / sizeof(T);
            unsigned char* ib = ibuf + kp * (Img::kBufChunks * 16);        // this tile's image buffer
            cp_async_wait_all();
            __syncwarp();
            if constexpr (kBits) {                                       // E1, first half: the block's set bits -> raw IDs in the slot
                if (!listed) bm_expand<T, kLandChunks>(reinterpret_cast<T*>(slot), s_start[k & (kRing - 1)], warp, q, l, land, a.bitmap, a.id_base);
                __syncwarp();
            }
            uint32_t d[32];
            bool wide_lane = false, wide = false;
            const T base = col_deltas<W>(raw, m, d, wide_lane);          // E1
            if constexpr (W == 64 && !kBits) wide = __any_sync(kFull, wide_lane);   // (a bitmap of < 2^32 bits: every delta fits 32 bits)
            if (!wide) key = a.codec == BFSC_CODEC_BP128 ? quad_max_width_key(d) : quad_choose_b<W>(d);   // E2
            // The bulk store that read this image buffer (issued when the previous iteration ended) is done with it.
            // Not waited for before E2: the copy engine needs half a microsecond to fetch its source.
            if (lane == 0) bulk_wait_read();
            __syncwarp();
            if (wide) key = wide_choose_b(reinterpret_cast<const uint64_t*>(raw), m, reinterpret_cast<uint32_t*>(ib + q * (Img::kSlotChunks * 16)),
                                     a.codec == BFSC_CODEC_BP128);
            if (m <= 0) key = 0;
            if (l == 0) s_key[kp][j] = key;
            {   // The tile's aggregate goes out as soon as the LAST worker warp has its sizes — not when the scan
                // warp gets to it: that warp may still be inside an earlier tile's look-back, and every
                // later tile in flight waits for this number.
                uint32_t z = l == 0 ? key >> 18 : 0u;
                z += __shfl_xor_sync(kFull, z, 4); z += __shfl_xor_sync(kFull, z, 8); z += __shfl_xor_sync(kFull, z, 16);
                if (lane == 0) {
                    const unsigned int old = atomicAdd(&s_agg[k & 3], (1u << 24) | z);
                    if ((old >> 24) == kEncWorkers - 1) {
                        s_agg[k & 3] = 0;
                        const unsigned long long t = s_tile[k & (kRing - 1)];
                        pdl_wait();                                      // the states are zeroed by the plan kernel
                        if (t > 0)
                            st_volatile_u64(&a.ws.tile_state[t * kStateStride], kFlagAgg | (unsigned long long)((old & 0xffffffu) + z));
                    }
                }
            }
            bar_arrive(kBarSizes + kp, kSizesThreads);

            const uint32_t b = 64u - ((key >> 7) & 127u), n_exc = key & 127u;
            // u64 ID arrays: a block whose deltas fit 32 bits but whose image does not fit its slot (b > 17: gaps over 2^17)
            // is packed from the registers STRAIGHT to its place in the output — this tile's offsets are awaited first
            // (the scan warp needs only the sizes, posted above), which costs this warp its one tile of slack, not a
            // re-read of the IDs with 64-bit arithmetic (late_emit: 2^24 IDs with gaps of 2^20 took 187 us, the same
            // IDs with gaps of 16 take 49).
            bool direct = false;
            if constexpr (W == 64 && !kBits) direct = !wide && key != 0 && (key >> 14) > (uint32_t)Img::kCap;
            const bool late = !kBits && key != 0 && !direct && (wide || (key >> 14) > (uint32_t)Img::kCap);   // slow path, in global memory later
            const bool fast = !wide && key != 0 && !late && !direct;
            // The warp's 8 images lie back to back in the buffer, as they do in the output (consecutive blocks):
            // woff = exclusive scan of the fast blocks' sizes over the quads, in 16-byte chunks.
            {
                const uint32_t zf = fast ? key >> 18 : 0u;
                uint32_t inc = zf, y;
                y = __shfl_up_sync(kFull, inc, 4); if (lane >= 4) inc += y;
                y = __shfl_up_sync(kFull, inc, 8); if (lane >= 8) inc += y;
                y = __shfl_up_sync(kFull, inc, 16); if (lane >= 16) inc += y;
                woff = inc - zf;
            }
            unsigned char* img = ib + 16 * woff;
            BFSC_CHECK(!fast || 16u * woff + (key >> 14) <= (uint32_t)(Img::kBufChunks * 16));
            bool emit = fast;                                            // this quad packs now (into the image buffer, or directly)
            if constexpr (W == 64 && !kBits) {
                if (__any_sync(kFull, direct)) {
                    mbar_wait(&mb_off[kp], (k / kNB) & 1);               // this tile's offsets are resolved
                    if (direct) {
                        const unsigned long long at = s_at[kp][j];
                        emit = at != kSkip;                              // (kSkip: over the output capacity, status is set)
                        img = a.out + at;
                        BFSC_CHECK(!emit || at + (key >> 14) <= a.out_cap);
                    }
                }
            }
            if (!wide && __any_sync(kFull, emit && n_exc > 0))           // E4 into the image buffer: exceptions
                col_exceptions_raw<W>(d, raw, img + 16 + 16 * b, b, emit ? n_exc : 0u);
            __syncwarp();                                                // the warp's staged IDs are consumed
            mbar_wait(&mb_post[(k + 1) & (kRing - 1)], ((k + 1) / kRing) & 1);   // tile k+1 is posted
            have_next = s_tile[(k + 1) & (kRing - 1)] != kNoTile;
            if constexpr (kBits) {
                if (have_next) {
                    if (listed) quad_prefetch<W>(slot, list + blk_xoff((k + 1) & (kRing - 1), j), blk_m((k + 1) & (kRing - 1), j));
                    else bm_prefetch<kLandChunks>(land, a.bitmap, s_start[(k + 1) & (kRing - 1)], warp, lane);
                }
            } else {
                if (have_next) quad_prefetch<W>(slot, ids + blk_xoff((k + 1) & (kRing - 1), j), blk_m((k + 1) & (kRing - 1), j));   // same slots
            }
            if (emit) {                                                  // payload + header
                if (b > 0) col_pack32(d, b, reinterpret_cast<uint32_t*>(img) + 4 + l);
                if (l == 0) {                                            // block header (FORMAT.md §2)
                    reinterpret_cast<unsigned long long*>(img)[0] = (unsigned long long)base;
                    reinterpret_cast<unsigned long long*>(img)[1] = (unsigned long long)(b | (n_exc << 8));
                }
            }
            if (late) key |= kLateBit;
            if (direct) key |= kDoneBit;                                 // nothing of it waits in shared memory (and the warp's images are not one piece)
            __syncwarp();                                                // image complete
            n_wait++;
        }

        // copy out the oldest waiting tile: tile k - kDefer while tiles keep coming, then drain
        const int w = n_wait - (have ? 1 : 0);                           // waiting tiles older than tile k
        if (w > 0 && (w == kDefer || !have)) {
            const uint32_t key_e = (kDefer == 2 && w == 2) ? key_hist[kDefer - 1] : key_hist[0];     // key and image place
            const uint32_t woff_e = (kDefer == 2 && w == 2) ? woff_hist[kDefer - 1] : woff_hist[0];  // of the CTA's tile ke
            int kpe = kp - w;                                            // its buffer: ke % kNB
            if (kpe < 0) kpe += kNB;
            mbar_wait(&mb_off[kpe], (ke / kNB) & 1);                     // its offsets are resolved
            unsigned long long at = kSkip;
            if (key_e != 0) at = s_at[kpe][j];
            if (__any_sync(kFull, (key_e & kLateBit) != 0)) {
                const bool mine = (key_e & kLateBit) != 0 && at != kSkip;
                if constexpr (!kBits) late_emit<W>(ids + blk_xoff(ke & (kRing - 1), j), blk_m(ke & (kRing - 1), j), key_e & ~kLateBit, mine ? a.out + at : nullptr);
            }
            // images -> their final place. Usual case: the warp's blocks are consecutive in the output as well
            // (same stream, none late, all fit): ONE bulk store of the whole buffer by lane 0.
            const unsigned char* ib_e = ibuf + kpe * (Img::kBufChunks * 16);
            const bool valid = key_e != 0, fast_e = valid && (key_e & (kLateBit | kDoneBit)) == 0;
            const uint32_t z_e = fast_e ? key_e >> 18 : 0u;
            const unsigned long long at_n = __shfl_down_sync(kFull, at, 4);
            const bool valid_n = __shfl_down_sync(kFull, (int)valid, 4) != 0 && q < kQuadBlocks - 1;
            const bool contig = !valid || (fast_e && at != kSkip && (!valid_n || at_n == at + 16ull * z_e));
            if (__all_sync(kFull, contig)) {
                const uint32_t tot = __shfl_sync(kFull, woff_e + z_e, 31);
                fence_proxy_async_smem();                                // the image was written through the generic proxy
                __syncwarp();
                BFSC_CHECK(lane != 0 || tot == 0 || (at + 16ull * tot <= a.out_cap && 16u * tot <= (uint32_t)(Img::kBufChunks * 16)));
                if (lane == 0 && tot > 0) bulk_store(a.out + at, ib_e, 16u * tot);
            } else if (fast_e && at != kSkip) {
                const uint4* src = reinterpret_cast<const uint4*>(ib_e) + woff_e;
                uint4* dst = reinterpret_cast<uint4*>(a.out + at);
                BFSC_CHECK(at + 16ull * z_e <= a.out_cap);
                for (uint32_t c = l; c < z_e; c += 4) __stcs(dst + c, src[c]);
            }
            __syncwarp();
            n_wait--;
            ke++;
        }
        if (!have && n_wait == 0) break;
        if (have) {
#pragma unroll
            for (int x = kDefer - 1; x > 0; x--) { key_hist[x] = key_hist[x - 1]; woff_hist[x] = woff_hist[x - 1]; }
            key_hist[0] = key; woff_hist[0] = woff;
            kp = kp == kNB - 1 ? 0 : kp + 1;
        }
        have = have_next;
    }
    if (lane == 0) bulk_wait_all();                                      // the bulk stores have left shared memory and landed
}

// E5 by one warp: y[0 .. padded) = x[0 .. n), zeros behind. Eight loads in flight per lane (a plain loop waits for every
// load before it issues the next: a 1 KB RAW stream then costs eight round trips to L2).
template <typename T>
__device__ __forceinline__ void raw_copy(T* __restrict__ y, const T* __restrict__ x, unsigned long long n, unsigned long long padded, int lane) {
    for (unsigned long long t0 = 0; t0 < padded; t0 += 32 * 8) {
        T v[8];
#pragma unroll
        for (int u = 0; u < 8; u++) { const unsigned long long t = t0 + 32 * u + lane; v[u] = t < n ? x[t] : (T)0; }
#pragma unroll
        for (int u = 0; u < 8; u++) { const unsigned long long t = t0 + 32 * u + lane; if (t < padded) y[t] = v[u]; }
    }
}

// ---- stream headers, directory tails, E5 raw passthrough, out_offsets (batch / degenerate calls) ----
template <int W>
__global__ void __launch_bounds__(256) k_enc_streams(EncArgs a) {
    using T = typename IdT<W>::T;
    constexpr unsigned long long E = W / 8;
    pdl_wait();
    pdl_launch_dependents();
    const unsigned long long total_blocks = a.ws.hdr->total_blocks, grand16 = a.ws.hdr->grand16;
    bool ok = a.ws.hdr->ok != 0;
    if (ok && a.ws.hdr->total_out > a.out_cap) {
        ok = false;
        if (blockIdx.x == 0 && threadIdx.x == 0) set_status(a.status, BFSC_ERR_DST_TOO_SMALL);
    }
    // byte offset of stream i = fixed_prefix[i] + 16 * (scan value at its first block q). The block belongs to
    // stream i itself when the stream has blocks (q_next > q: no search, one load less in the chain), else to
    // the next stream that has some.
    // ss_i / fp_i: stream_start[i] and fixed_prefix[i], requested by the caller together with the block counts (a stream
    // with blocks — the usual case — then needs no further load: one round trip per buffer instead of three)
    auto stream_at = [&](uint32_t i, unsigned long long q, unsigned long long q_next, unsigned long long ss_i, unsigned long long fp_i) -> unsigned long long {
        unsigned long long bb = grand16;
        if (q < total_blocks) {
            if (q_next > q) bb = (ss_i - 1 - fp_i) >> 4;
            else {
                const uint32_t j = a.in_off ? find_buf_from(a.ws.blk_first, a.n_buf, q, group_hint(a.ws.tile_state, q)) : 0u;
                bb = (a.ws.stream_start[j] - 1 - a.ws.fixed_prefix[j]) >> 4;
            }
        }
        return fp_i + 16ull * bb;
    };
    const int lane = threadIdx.x & 31, warps = blockDim.x >> 5;
    for (uint32_t i = blockIdx.x * warps + (threadIdx.x >> 5); i < a.n_buf; i += gridDim.x * warps) {   // warp = buffer
        const unsigned long long f0 = a.ws.blk_first[i], f1 = a.ws.blk_first[i + 1];
        const unsigned long long f2 = (i + 1 < a.n_buf) ? a.ws.blk_first[i + 2] : f1;
        const unsigned long long ss0 = a.ws.stream_start[i], ss1 = a.ws.stream_start[i + 1];
        const unsigned long long fp0 = a.ws.fixed_prefix[i], fp1 = a.ws.fixed_prefix[i + 1];
        if (!ok) { if (lane == 0) { if (a.out_off) a.out_off[i] = 0; if (a.out_sizes) a.out_sizes[i] = 0; } continue; }
        const unsigned long long s0 = stream_at(i, f0, f1, ss0, fp0);
        const unsigned long long s1 = (i + 1 < a.n_buf) ? stream_at(i + 1, f1, f2, ss1, fp1) : a.ws.hdr->total_out;
        const unsigned long long n = buf_count(a, i), total = s1 - s0;
        const bool raw = n * E < a.thr;
        unsigned char* s = a.out + s0;
        if (a.dst) {                                                      // scatter call: the stream has its own destination
            const unsigned long long d = a.dst[i];
            const bool fits = d != 0 && !(d & 15) && total <= a.dst_cap;
            if (lane == 0) {
                a.out_sizes[i] = fits ? total : 0ull;
                if (!fits) set_status(a.status, (d == 0 || (d & 15)) ? BFSC_ERR_INVALID_ARG : BFSC_ERR_DST_TOO_SMALL);
            }
            if (!fits) continue;
            s = reinterpret_cast<unsigned char*>(d);
        }
        if (lane == 0) {
            if (a.out_off) a.out_off[i] = s0;
            const unsigned long long nb = f1 - f0;
            uint4 h0, h1;
            h0.x = 0x43534642u;                                           // "BFSC"
            h0.y = 1u | ((uint32_t)W << 8) | ((raw ? 0u : a.codec) << 16);
            h0.z = (uint32_t)n; h0.w = (uint32_t)(n >> 32);
            h1.x = (uint32_t)total; h1.y = (uint32_t)(total >> 32);
            h1.z = (uint32_t)nb; h1.w = 0;
            reinterpret_cast<uint4*>(s)[0] = h0;
            reinterpret_cast<uint4*>(s)[1] = h1;
            if (!raw) {                                                   // dir[nb] and the zero pad
                uint32_t* dir = reinterpret_cast<uint32_t*>(s + 32);
                dir[nb] = (uint32_t)(total >> 4);
                for (unsigned long long q = nb + 1; q < ((nb + 1 + 3) & ~3ull); q++) dir[q] = 0;
            }
        }
        if (raw) {                                                        // E5: verbatim copy + zero pad
            const T* x = reinterpret_cast<const T*>(a.ids) + buf_start(a, i);
            T* y = reinterpret_cast<T*>(s + 32);
            const unsigned long long padded = (total - 32) / E;
            raw_copy<T>(y, x, n, padded, lane);
        }
    }
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        const unsigned long long t = ok ? a.ws.hdr->total_out : 0ull;
        if (a.out_off) a.out_off[a.n_buf] = t;
        if (a.out_total) *a.out_total = t;
    }
}

// ---- Small batches (a BFS level of up to ~1 MB): the WHOLE compress call in one launch of one thread-block cluster ----
// kSmallCtas CTAs that the hardware schedules together, so that a CTA may wait for another one of the grid without any
// residency assumption, and that exchange their tile sums through distributed shared memory instead of a look-back
// through L2. Every CTA runs E0 for itself (the plan of up to kSmallMaxBuf buffers, tables in shared memory), then
//   pass 1   E1 + E2 of its tiles (tile T = kSmallCtas r + cluster rank, r = 0 .. kSmallIters - 1): sizes in shared memory; the
//            scan inside each own tile and its sum written into every CTA of the cluster;   -- ONE cluster barrier --
//            exclusive scan of the <= 32 tile sums (every CTA the same): every CTA now has the output offset of every
//            block and every stream of the batch in its own shared memory;
//   pass 2   E1 + E4 of its tiles (IDs staged again if there are several: they come from L2), blocks and directory
//            entries written to their final place; stream headers, directory tails, RAW copies (E5), out_offsets
//            of its share of the streams.
// No plan kernel, no look-back states, no ticket, no k_enc_streams: one launch latency instead of three.
constexpr int kSmallCtas = 16;                           // CTAs of the cluster (above the portable 8: opt-in, checked once per device)
constexpr int kSmallIters = 2;                           // tiles per CTA (measured: with 4 the general path is faster from 3 tiles on)
constexpr uint32_t kSmallMaxBuf = 1024;
constexpr uint32_t kSmallMaxBlocks = kSmallCtas * kTileR * kSmallIters;      // 2048 blocks = 262144 IDs
static_assert(kSmallCtas * kSmallIters <= 32, "one warp scans the tile sums");
constexpr int kSmallThreads = kEncWorkers * 32;

template <int W> struct SmallSmem {
    static constexpr int kStageChunks = RawCfg<W>::kAreaChunks;              // per warp: staged raw IDs
    static constexpr int kSlotChunks = 34;                                   // per quad: one block image (every block with 32-bit deltas fits: 16 + 16 * 32 + 16)
    static constexpr int kWarpChunks = kStageChunks + kQuadBlocks * kSlotChunks;
    static constexpr size_t kBytes = (size_t)kEncWorkers * kWarpChunks * 16;
};

__device__ __forceinline__ uint32_t cluster_ctarank() {
    uint32_t r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
    return r;
}
__device__ __forceinline__ void cluster_sync_all() {     // every thread of every CTA of the cluster; orders shared AND global memory
    asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}
__device__ __forceinline__ void st_cluster_u32(uint32_t* local_ptr, uint32_t rank, uint32_t v) {   // the same variable in CTA `rank` of the cluster
    const uint32_t la = (uint32_t)__cvta_generic_to_shared(local_ptr);
    uint32_t ra;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(ra) : "r"(la), "r"(rank));
    asm volatile("st.shared::cluster.u32 [%0], %1;" ::"r"(ra), "r"(v) : "memory");
}

template <int W>
__global__ void __launch_bounds__(kSmallThreads, 1) k_enc_small(EncArgs a) {
    using T = typename IdT<W>::T;
    using Smem = SmallSmem<W>;
    constexpr unsigned long long E = W / 8;
    extern __shared__ __align__(16) uint4 dyn_smem[];
    __shared__ uint32_t s_first[kSmallMaxBuf + 1];                   // first block of every buffer (entry n_buf: total)
    __shared__ unsigned long long s_fixed[kSmallMaxBuf + 1];         // exclusive prefix of the fixed bytes
    __shared__ uint32_t s_key[kSmallIters][kTileR];                  // size<<14 | (64-b)<<7 | n_exc (| kLateBit), 0 = no block
    __shared__ uint32_t s_off16[kSmallCtas * kSmallIters][kTileR];   // exclusive scan of the sizes inside EVERY tile of the cluster (16-B units; tile T = block / 64), each row written by its CTA
    __shared__ uint32_t s_buf[kSmallIters][kTileR];                  // buffer, valid IDs, first ID (element) of every own block
    __shared__ int s_m[kSmallIters][kTileR];
    __shared__ unsigned long long s_xoff[kSmallIters][kTileR];
    __shared__ uint32_t s_sum[kSmallIters];                          // sums of the own tiles
    __shared__ uint32_t s_tsum[kSmallCtas * kSmallIters];            // sums of ALL tiles (written by their CTAs), then their exclusive scan
    __shared__ Scan2 sm[33];
    __shared__ int bad;
    pdl_wait();                                                      // the call before this one is complete (workspace, inputs)
    pdl_launch_dependents();
    const uint32_t rank = cluster_ctarank();
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, q = lane >> 2, l = lane & 3;
    const T* ids = reinterpret_cast<const T*>(a.ids);

    // ---- E0, by every CTA for itself
    if (threadIdx.x == 0) bad = 0;
    if (threadIdx.x < kSmallIters) s_sum[threadIdx.x] = 0;
    __syncthreads();
    auto zero_outputs = [&]() {                                      // an error of the whole call: every offset / size reads 0
        for (uint32_t i = rank * kSmallThreads + threadIdx.x; i <= a.n_buf; i += kSmallCtas * kSmallThreads) {
            if (a.out_off) a.out_off[i] = 0;
            if (a.out_sizes && i < a.n_buf) a.out_sizes[i] = 0;
        }
    };
    {
        constexpr int kIpt = kSmallMaxBuf / kSmallThreads;           // 4
        Scan2 v[kIpt], sum{0, 0};
#pragma unroll
        for (int u = 0; u < kIpt; u++) {
            const uint32_t i = threadIdx.x * kIpt + u;
            v[u] = Scan2{0, 0};
            if (i < a.n_buf) {
                const unsigned long long o0 = a.in_off[i], o1 = a.in_off[i + 1];
                if (o1 < o0) bad = 1;
                const unsigned long long n = o1 - o0;
                const bool raw = n * E < a.thr;                      // FORMAT.md §1 (L1311)
                const unsigned long long nb = raw ? 0ull : (n + kBlk - 1) / kBlk;
                v[u].a = nb;
                v[u].b = raw ? 32ull + ((n * E + 15ull) & ~15ull) : 32ull + ((4ull * (nb + 1) + 15ull) & ~15ull);
            }
            sum.a += v[u].a; sum.b += v[u].b;
        }
        Scan2 tot;
        Scan2 ex = block_scan_excl2(sum, &tot, sm);
#pragma unroll
        for (int u = 0; u < kIpt; u++) {
            const uint32_t i = threadIdx.x * kIpt + u;
            if (i < a.n_buf) { s_first[i] = (uint32_t)min(ex.a, 0xffffffffull); s_fixed[i] = ex.b; }
            ex.a += v[u].a; ex.b += v[u].b;
        }
        if (threadIdx.x == 0) { s_first[a.n_buf] = (uint32_t)min(tot.a, 0xffffffffull); s_fixed[a.n_buf] = tot.b; }
        __syncthreads();
        if (bad || tot.a > a.ws.blk_cap || tot.a > kSmallMaxBlocks) {        // (the same decision in every CTA of the cluster)
            if (rank == 0 && threadIdx.x == 0) set_status(a.status, BFSC_ERR_INVALID_ARG);
            zero_outputs();
            return;
        }
    }
    const uint32_t total = s_first[a.n_buf];
    const int R = (int)((total + kSmallCtas * kTileR - 1) / (kSmallCtas * kTileR));      // tiles per CTA that hold blocks
    uint4* area = dyn_smem + warp * Smem::kWarpChunks;
    uint4* slot = area + raw_slot_chunk<W>(q);
    unsigned char* img = reinterpret_cast<unsigned char*>(area + Smem::kStageChunks) + q * (Smem::kSlotChunks * 16);
    const int j = warp * kQuadBlocks + q;                            // the quad's block inside a tile

    // ---- pass 1: E1 + E2
    for (int r = 0; r < R; r++) {
        const uint32_t g = (uint32_t)r * (kSmallCtas * kTileR) + rank * kTileR + (uint32_t)j;
        int m = 0; uint32_t i = 0; unsigned long long xoff = 0;
        if (g < total) {
            i = bisect_first(s_first, a.n_buf, g);
            const unsigned long long o0 = a.in_off[i], n = a.in_off[i + 1] - o0, k = g - s_first[i];
            m = (int)min((unsigned long long)kBlk, n - kBlk * k);
            xoff = o0 + kBlk * k;
        }
        if (l == 0) { s_buf[r][j] = i; s_m[r][j] = m; s_xoff[r][j] = xoff; }
        quad_prefetch<W>(slot, ids + xoff, m);
        cp_async_wait_all();
        __syncwarp();
        const T* raw = reinterpret_cast<const T*>(slot) + (reinterpret_cast<uintptr_t>(ids + xoff) & 15) / sizeof(T);
        uint32_t d[32];
        bool wide_lane = false, wide = false;
        col_deltas<W>(raw, m, d, wide_lane);
        if constexpr (W == 64) wide = __any_sync(kFull, wide_lane);
        uint32_t key;
        if (!wide) key = a.codec == BFSC_CODEC_BP128 ? quad_max_width_key(d) : quad_choose_b<W>(d);
        else key = wide_choose_b(reinterpret_cast<const uint64_t*>(raw), m, reinterpret_cast<uint32_t*>(img), a.codec == BFSC_CODEC_BP128);
        if (m <= 0) key = 0;
        const bool late = key != 0 && (wide || (key >> 14) > (uint32_t)(Smem::kSlotChunks * 16));
        if (l == 0) s_key[r][j] = key | (late ? kLateBit : 0u);
        uint32_t z = l == 0 ? key >> 18 : 0u;
        z += __shfl_xor_sync(kFull, z, 4); z += __shfl_xor_sync(kFull, z, 8); z += __shfl_xor_sync(kFull, z, 16);
        if (lane == 0) atomicAdd(&s_sum[r], z);
        __syncwarp();                                                // the staged IDs are consumed (the next tile overwrites them)
    }
    __syncthreads();
    // ---- E3. Warp r: exclusive scan of the 64 sizes of own tile r (tile T = kSmallCtas r + rank = first block / 64); the row and the
    // tile's sum go into EVERY CTA of the cluster (distributed shared memory), so that after ONE cluster barrier every CTA
    // knows the scan value at every block of the batch: no look-back, no exchange through global memory.
    if (warp < R) {
        const int r = warp, Tl = r * kSmallCtas + (int)rank;
        const uint32_t k0 = s_key[r][2 * lane] & ~kLateBit, k1 = s_key[r][2 * lane + 1] & ~kLateBit;
        const uint32_t own = (k0 >> 18) + (k1 >> 18);
        uint32_t inc = own;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { const uint32_t y = __shfl_up_sync(kFull, inc, o); if (lane >= o) inc += y; }
        const uint32_t e0 = inc - own, e1 = e0 + (k0 >> 18), sum = __shfl_sync(kFull, inc, 31);
#pragma unroll
        for (int c = 0; c < kSmallCtas; c++) {
            st_cluster_u32(&s_off16[Tl][2 * lane], (uint32_t)c, e0);
            st_cluster_u32(&s_off16[Tl][2 * lane + 1], (uint32_t)c, e1);
            if (lane == 0) st_cluster_u32(&s_tsum[Tl], (uint32_t)c, sum);
        }
    }
    cluster_sync_all();
    if (warp == 0) {                                                 // exclusive scan of the tile sums (tiles beyond the last block: never written, never read)
        const int nT = R * kSmallCtas;
        const uint32_t v = lane < nT ? s_tsum[lane] : 0u;
        uint32_t inc = v;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { const uint32_t y = __shfl_up_sync(kFull, inc, o); if (lane >= o) inc += y; }
        if (lane < nT) s_tsum[lane] = inc - v;
        if (lane == 31) s_sum[0] = inc;                              // grand total (16-B units); the own sums are no longer needed
    }
    __syncthreads();
    const unsigned long long grand16 = s_sum[0];
    const unsigned long long total_out = s_fixed[a.n_buf] + 16ull * grand16;
    if (total_out > a.out_cap) {                                     // (the same decision in every CTA)
        if (rank == 0 && threadIdx.x == 0) set_status(a.status, BFSC_ERR_DST_TOO_SMALL);
        zero_outputs();
        return;
    }
    auto dst_ok = [&](unsigned long long d, unsigned long long stream_bytes) -> bool {   // scatter calls: a usable destination that holds the stream
        return d != 0 && !(d & 15) && stream_bytes <= a.dst_cap;
    };
    // scan value at block g: 16-B units of block bytes before it (g = total: all of them)
    auto scan_at = [&](uint32_t g) -> unsigned long long {
        return g >= total ? grand16 : (unsigned long long)s_tsum[g / kTileR] + s_off16[g / kTileR][g % kTileR];
    };
    // stream i starts at fixed_prefix[i] + 16 * (scan value at its first block; streams without blocks: at the next block)
    auto stream_at = [&](uint32_t i) -> unsigned long long {
        return i >= a.n_buf ? total_out : s_fixed[i] + 16ull * scan_at(s_first[i]);
    };

    // ---- pass 2: E1 + E4, blocks and directory entries to their final place
    for (int r = 0; r < R; r++) {
        const uint32_t g = (uint32_t)r * (kSmallCtas * kTileR) + rank * kTileR + (uint32_t)j;
        const int m = s_m[r][j];
        const uint32_t i = s_buf[r][j];
        const unsigned long long xoff = s_xoff[r][j];
        if (R > 1) {                                                 // (R == 1: the tile is still staged)
            quad_prefetch<W>(slot, ids + xoff, m);
            cp_async_wait_all();
            __syncwarp();
        }
        const T* raw = reinterpret_cast<const T*>(slot) + (reinterpret_cast<uintptr_t>(ids + xoff) & 15) / sizeof(T);
        const uint32_t stored = s_key[r][j], key = stored & ~kLateBit;
        const bool late = (stored & kLateBit) != 0, fast = key != 0 && !late;
        const uint32_t b = 64u - ((key >> 7) & 127u), n_exc = key & 127u;
        unsigned long long at = 0;
        bool placed = key != 0;                                      // (scatter calls: and the stream fits its destination)
        if (key != 0) {
            at = s_fixed[i + 1] + 16ull * scan_at(g);
            unsigned long long S = stream_at(i);
            if (a.dst) {                                             // the stream has its own destination: `at` becomes an address
                const unsigned long long dsti = a.dst[i];
                placed = dst_ok(dsti, stream_at(i + 1) - S);
                at = dsti + (at - S);
                S = dsti;
            }
            if (l == 0 && placed)                                    // directory entry (FORMAT.md §1)
                reinterpret_cast<uint32_t*>(a.out + S + 32)[g - s_first[i]] = (uint32_t)((at - S) >> 4);
        }
        uint32_t d[32];
        bool wide_lane = false;
        const T base = col_deltas<W>(raw, m, d, wide_lane);
        if (__any_sync(kFull, fast && n_exc > 0)) col_exceptions_raw<W>(d, raw, img + 16 + 16 * b, b, fast ? n_exc : 0u);
        if (fast) {
            if (b > 0) col_pack32(d, b, reinterpret_cast<uint32_t*>(img) + 4 + l);
            if (l == 0) {                                            // block header (FORMAT.md §2)
                reinterpret_cast<unsigned long long*>(img)[0] = (unsigned long long)base;
                reinterpret_cast<unsigned long long*>(img)[1] = (unsigned long long)(b | (n_exc << 8));
            }
        }
        __syncwarp();
        BFSC_CHECK(key == 0 || at + (key >> 14) <= a.out_cap);
        BFSC_CHECK(!fast || (key >> 14) <= (uint32_t)(Smem::kSlotChunks * 16));
        if (fast && placed) {
            const uint4* src = reinterpret_cast<const uint4*>(img);
            uint4* dst = reinterpret_cast<uint4*>(a.out + at);
            for (uint32_t c = l; c < (key >> 18); c += 4) __stcs(dst + c, src[c]);
        }
        if (__any_sync(kFull, late)) late_emit<W>(ids + xoff, m, key, late && placed ? a.out + at : nullptr);
        __syncwarp();                                                // image and staged IDs are free again
    }

    if (a.n_buf == 0 && rank == 0 && threadIdx.x == 0 && a.out_off) a.out_off[0] = total_out;
    // ---- stream headers, directory tails, E5 (RAW copies), out_offsets: a warp per stream, the streams dealt round the cluster
    for (uint32_t i = rank * kEncWorkers + warp; i < a.n_buf; i += kSmallCtas * kEncWorkers) {
        const unsigned long long s0 = stream_at(i), s1 = stream_at(i + 1);
        BFSC_CHECK(s0 + 32 <= s1 && s1 <= a.out_cap);
        const unsigned long long o0 = a.in_off[i], n = a.in_off[i + 1] - o0, tot = s1 - s0;
        if (lane == 0 && a.out_off) { a.out_off[i] = s0; if (i + 1 == a.n_buf) a.out_off[a.n_buf] = s1; }
        const bool raw_s = n * E < a.thr;
        unsigned char* s = a.out + s0;
        if (a.dst) {
            const unsigned long long dsti = a.dst[i];
            const bool fits = dst_ok(dsti, tot);
            if (lane == 0) {
                a.out_sizes[i] = fits ? tot : 0ull;
                if (!fits) set_status(a.status, (dsti == 0 || (dsti & 15)) ? BFSC_ERR_INVALID_ARG : BFSC_ERR_DST_TOO_SMALL);
            }
            if (!fits) continue;
            s = reinterpret_cast<unsigned char*>(dsti);
        }
        if (lane == 0) {
            const unsigned long long nb = s_first[i + 1] - s_first[i];
            uint4 h0, h1;
            h0.x = 0x43534642u;                                      // "BFSC"
            h0.y = 1u | ((uint32_t)W << 8) | ((raw_s ? 0u : a.codec) << 16);
            h0.z = (uint32_t)n; h0.w = (uint32_t)(n >> 32);
            h1.x = (uint32_t)tot; h1.y = (uint32_t)(tot >> 32);
            h1.z = (uint32_t)nb; h1.w = 0;
            reinterpret_cast<uint4*>(s)[0] = h0;
            reinterpret_cast<uint4*>(s)[1] = h1;
            if (!raw_s) {                                            // dir[nb] and the zero pad
                uint32_t* dir = reinterpret_cast<uint32_t*>(s + 32);
                dir[nb] = (uint32_t)(tot >> 4);
                for (unsigned long long x = nb + 1; x < ((nb + 1 + 3) & ~3ull); x++) dir[x] = 0;
            }
        }
        if (raw_s) {                                                 // E5: verbatim copy + zero pad
            const T* x = ids + o0;
            T* y = reinterpret_cast<T*>(s + 32);
            const unsigned long long padded = (tot - 32) / E;
            raw_copy<T>(y, x, n, padded, lane);
        }
    }
}

// ---- FORMAT.md §8: RAW fallback of a single-buffer call (ID array source). After the stream is complete (its size is
// in ws.hdr->total_out): if it is not smaller than the RAW stream of the same IDs, it is overwritten by that one
// (header, verbatim IDs, zero pad) and *out_total follows. The input is read a second time only then.
template <int W>
__global__ void __launch_bounds__(256) k_enc_fallback(EncArgs a) {
    using T = typename IdT<W>::T;
    constexpr unsigned long long E = W / 8;
    pdl_wait();
    pdl_launch_dependents();
    const unsigned long long n = a.n_single, body = (n * E + 15ull) & ~15ull, raw_total = 32ull + body;
    if (a.ws.hdr->ok == 0 || n * E < a.thr) return;                          // RAW already (by the threshold)
    const unsigned long long have = a.ws.hdr->total_out;
    if (have > a.out_cap || have < raw_total) return;                        // (an error was flagged) | smaller: keep
    const T* x = reinterpret_cast<const T*>(a.ids);
    T* y = reinterpret_cast<T*>(a.out + 32);
    const unsigned long long padded = body / E;
    for (unsigned long long j = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; j < padded;
         j += (unsigned long long)gridDim.x * blockDim.x)
        y[j] = j < n ? x[j] : (T)0;
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        uint4 h0, h1;
        h0.x = 0x43534642u; h0.y = 1u | ((uint32_t)W << 8);                  // mode 0
        h0.z = (uint32_t)n; h0.w = (uint32_t)(n >> 32);
        h1.x = (uint32_t)raw_total; h1.y = (uint32_t)(raw_total >> 32); h1.z = 0; h1.w = 0;
        reinterpret_cast<uint4*>(a.out)[0] = h0;
        reinterpret_cast<uint4*>(a.out)[1] = h1;
        if (a.out_total) *a.out_total = raw_total;
    }
}

// ---- FORMAT.md §9: a frontier bitmap as the source. Chunk = 32 words = 1024 bits.
constexpr int kChunkBits = 1024;

constexpr int kSuperChunks = 32;                         // chunks per super-chunk: one warp counts one super-chunk (4 KB of bitmap)
__device__ __forceinline__ uint32_t bm_word(const EncArgs& a, unsigned long long c, int lane) {   // word `lane` of chunk c, bits >= n_bits cleared
    const unsigned long long bit0 = c * kChunkBits + 32ull * lane;
    uint32_t x = bit0 < a.n_bits ? a.bitmap[c * 32 + lane] : 0u;
    if (bit0 < a.n_bits && a.n_bits - bit0 < 32) x &= (1u << (uint32_t)(a.n_bits - bit0)) - 1u;
    return x;
}
// Position of the k-th (k = 0: lowest) set bit of x; x has more than k set bits. Five halving steps.
__device__ __forceinline__ uint32_t select_bit(uint32_t x, uint32_t k) {
    uint32_t pos = 0;
#pragma unroll
    for (int w = 16; w > 0; w >>= 1) {
        const uint32_t c = (uint32_t)__popc(x & ((1u << w) - 1u));
        if (k >= c) { k -= c; x >>= w; pos += w; }
    }
    return pos;
}

// Set bits of every chunk -> a.chunk[c] (plain counts; entries up to the end of the last super-chunk: 0) and of every
// super-chunk -> a.super[s]. A CTA takes a super-chunk at a time (8 warps x 4 chunks), eight lanes per chunk, one 16-byte
// load each (the bitmap is 16-byte aligned and readable up to a multiple of 16 bytes).
__global__ void __launch_bounds__(256) k_bm_count(EncArgs a) {
    __shared__ uint32_t s_w[8];
    pdl_wait();                                          // the call before this one is complete (workspace, inputs)
    pdl_launch_dependents();
    const int lane = threadIdx.x & 31, sub = lane & 7, warp = threadIdx.x >> 5;
    for (unsigned long long sc = blockIdx.x; sc < a.n_super; sc += gridDim.x) {
        const unsigned long long c = sc * kSuperChunks + 4 * warp + (lane >> 3);
        const unsigned long long bit0 = c * kChunkBits + 128ull * sub;
        uint32_t k = 0;
        if (bit0 < a.n_bits) {
            const uint4 v = reinterpret_cast<const uint4*>(a.bitmap)[c * 8 + sub];
            const uint32_t w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
            for (int u = 0; u < 4; u++) {
                const unsigned long long b0 = bit0 + 32ull * u;
                uint32_t x = b0 < a.n_bits ? w[u] : 0u;
                if (b0 < a.n_bits && a.n_bits - b0 < 32) x &= (1u << (uint32_t)(a.n_bits - b0)) - 1u;
                k += (uint32_t)__popc(x);
            }
        }
        k += __shfl_xor_sync(kFull, k, 1); k += __shfl_xor_sync(kFull, k, 2); k += __shfl_xor_sync(kFull, k, 4);
        if (sub == 0) a.chunk[c] = k;
        const uint32_t kw = k + __shfl_xor_sync(kFull, k, 8);                    // the warp's four chunks
        const uint32_t kq = kw + __shfl_xor_sync(kFull, kw, 16);
        if (lane == 0) s_w[warp] = kq;
        __syncthreads();
        if (threadIdx.x == 0) a.super[sc] = (unsigned long long)s_w[0] + s_w[1] + s_w[2] + s_w[3] + s_w[4] + s_w[5] + s_w[6] + s_w[7];
        __syncthreads();
    }
}

// One CTA: block scan of the super-chunk totals, in place -> set bits before every super-chunk (entry n_super = n = the
// number of set bits); then the plan of the one stream (E0).
template <int W>
__global__ void __launch_bounds__(1024) k_bm_plan(EncArgs a) {
    __shared__ Scan2 sm[33];
    constexpr unsigned long long E = W / 8;
    pdl_wait();
    pdl_launch_dependents();
    Scan2 carry{0, 0};
    for (unsigned long long s0 = 0; s0 < a.n_super; s0 += 1024ull) {
        const unsigned long long sc = s0 + threadIdx.x;
        const unsigned long long mine = sc < a.n_super ? a.super[sc] : 0ull;
        Scan2 tot;
        const Scan2 ex = block_scan_excl2(Scan2{mine, 0}, &tot, sm);
        if (sc < a.n_super) a.super[sc] = carry.a + ex.a;
        carry.a += tot.a;
    }
    const unsigned long long n = carry.a;
    const bool raw = n * E < a.thr;
    const unsigned long long nb_all = (n + kBlk - 1) / kBlk, nb = raw ? 0ull : nb_all;
    const unsigned long long fixed = raw ? 32ull + ((n * E + 15ull) & ~15ull) : 32ull + ((4ull * (nb + 1) + 15ull) & ~15ull);
    const unsigned long long nt = (nb + kTileR - 1) / kTileR;
    const bool ok = nb_all + 1 <= a.ws.blk_cap && nt <= a.ws.tile_cap;
    if (ok)
        for (unsigned long long q = threadIdx.x; q < nt; q += blockDim.x) a.ws.tile_state[q * kStateStride] = 0;
    if (threadIdx.x == 0) {
        a.super[a.n_super] = n;
        a.ws.blk_first[0] = 0; a.ws.blk_first[1] = nb;
        a.ws.fixed_prefix[0] = 0; a.ws.fixed_prefix[1] = fixed;
        a.ws.stream_start[0] = 0; a.ws.stream_start[1] = 0;
        a.ws.hdr->total_blocks = nb; a.ws.hdr->fixed_total = fixed; a.ws.hdr->ticket = 0;
        a.ws.hdr->grand16 = 0; a.ws.hdr->total_out = fixed; a.ws.hdr->ok = ok ? 1u : 0u; a.ws.hdr->n_ids = n;
        if (!ok) set_status(a.status, BFSC_ERR_INVALID_ARG);
        if (a.out_total) *a.out_total = 0;               // (the last tile, or k_bm_finish, writes the size)
        if (ok && n == 0 && !raw) {                      // the empty stream (no tile runs; k_bm_finish is not launched when the
            if (48 <= a.out_cap) {                       //  call has neither a threshold nor the fallback option): 48 bytes
                uint4 h0, h1;
                h0.x = 0x43534642u; h0.y = 1u | ((uint32_t)W << 8) | (a.codec << 16); h0.z = 0; h0.w = 0;
                h1.x = 48u; h1.y = 0; h1.z = 0; h1.w = 0;
                reinterpret_cast<uint4*>(a.out)[0] = h0;
                reinterpret_cast<uint4*>(a.out)[1] = h1;
                reinterpret_cast<uint4*>(a.out)[2] = make_uint4(3u, 0u, 0u, 0u);
                if (a.out_total) *a.out_total = 48ull;
            } else set_status(a.status, BFSC_ERR_DST_TOO_SMALL);
        }
    }
}

// Where every block begins: starts[g] = bit index of the (128 g)-th set bit (u32, in ws.blk_tab), starts[nb_all] = n_bits.
// A warp takes kStartsPer chunks at a time: a chunk holds the block starts 128 g in [prefix, prefix + count), at most 8.
// The bitmap words (the caller's input, stable since this call's first kernel) are loaded and ranked BEFORE the wait for
// the plan kernel, all kStartsPer loads in flight at once; after it only the two prefix tables are read.
constexpr int kStartsPer = 4;
// Sparse bitmaps (at most one set bit in 16 on average, decided on the device from the popcount): no block starts — the IDs
// are written out as a list by the WHOLE grid here, a warp per chunk from the same chunk / super-chunk prefixes, and the tile
// kernel stages its blocks from that list as it does from an ID array. Inside the tile kernel a block's 128 set bits are
// found by ONE quad: a 0.2 % dense bitmap of 2^25 bits is 524 blocks of 2000 words each, 250 us on 9 CTAs while 139 SMs idle.
template <int W>
__global__ void __launch_bounds__(256) k_bm_starts(EncArgs a) {
    pdl_launch_dependents();
    const int lane = threadIdx.x & 31;
    const unsigned long long stride = (unsigned long long)gridDim.x * 8 * kStartsPer;
    unsigned long long c0 = ((unsigned long long)blockIdx.x * 8 + (threadIdx.x >> 5)) * kStartsPer;
    bool waited = false;
    for (; c0 < a.n_chunks; c0 += stride) {
        uint32_t x[kStartsPer], k[kStartsPer], inc[kStartsPer];
#pragma unroll
        for (int u = 0; u < kStartsPer; u++) x[u] = c0 + u < a.n_chunks ? bm_word(a, c0 + u, lane) : 0u;
#pragma unroll
        for (int u = 0; u < kStartsPer; u++) {
            k[u] = (uint32_t)__popc(x[u]);
            inc[u] = k[u];
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) { const uint32_t y = __shfl_up_sync(kFull, inc[u], o); if (lane >= o) inc[u] += y; }
        }
        if (!waited) { pdl_wait(); waited = true; }
        if (a.ws.hdr->ok == 0) return;
        const bool sparse = bm_sparse(a);
        // set bits before each of the warp's chunks: its super-chunk's prefix + the counts of the chunks before it in
        // the super-chunk (the warp's chunks share one: one coalesced load of its 32 counts, scanned here)
        unsigned long long p0[kStartsPer];
        {
            const unsigned long long sc = c0 / kSuperChunks;
            const uint32_t cnt = a.chunk[sc * kSuperChunks + lane];
            uint32_t ci = cnt;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) { const uint32_t y = __shfl_up_sync(kFull, ci, o); if (lane >= o) ci += y; }
            const unsigned long long sp = a.super[sc];
#pragma unroll
            for (int u = 0; u < kStartsPer; u++) p0[u] = sp + __shfl_sync(kFull, ci - cnt, (int)((c0 + u) % kSuperChunks));
        }
        if (sparse) {                                                // the ID list instead of block starts
            using T = typename IdT<W>::T;
            T* list = reinterpret_cast<T*>(a.list);
#pragma unroll
            for (int u = 0; u < kStartsPer; u++) {
                unsigned long long at = p0[u] + (inc[u] - k[u]);
                const unsigned long long id0 = a.id_base + (c0 + u) * kChunkBits + 32ull * lane;
                uint32_t xx = x[u];
                while (xx) {
                    const uint32_t b = (uint32_t)__ffs((int)xx) - 1u;
                    xx &= xx - 1u;
                    BFSC_CHECK(at < a.ws.hdr->n_ids);
                    list[at++] = (T)(id0 + b);
                }
            }
            continue;
        }
        uint32_t* starts = reinterpret_cast<uint32_t*>(a.ws.blk_tab);
#pragma unroll
        for (int u = 0; u < kStartsPer; u++) {
            // lane j takes the j-th block start of the chunk: rank r inside the chunk -> the word that holds it (the
            // number of words whose inclusive count is <= r: five shuffle steps) -> the bit inside that word
            const unsigned long long p1 = p0[u] + __shfl_sync(kFull, inc[u], 31);
            const unsigned long long g = (p0[u] + kBlk - 1) / kBlk + (unsigned)lane;
            const uint32_t r = (uint32_t)(g * kBlk - p0[u]);
            uint32_t pos = 0;
#pragma unroll
            for (int st = 16; st > 0; st >>= 1) {
                const uint32_t v = __shfl_sync(kFull, inc[u], (int)(pos + st - 1));
                if (v <= r) pos += st;
            }
            pos &= 31u;                                                  // (lanes beyond the chunk's last start: anything valid)
            const uint32_t xo = __shfl_sync(kFull, x[u], (int)pos);
            const uint32_t eo = __shfl_sync(kFull, inc[u] - k[u], (int)pos);
            if (g * kBlk < p1) starts[g] = (uint32_t)((c0 + u) * kChunkBits + 32ull * pos + select_bit(xo, r - eo));
        }
    }
    if (!waited) pdl_wait();
    if (blockIdx.x == 0 && threadIdx.x == 0 && a.ws.hdr->ok != 0 && !bm_sparse(a))
        reinterpret_cast<uint32_t*>(a.ws.blk_tab)[(a.ws.hdr->n_ids + kBlk - 1) / kBlk] = (uint32_t)a.n_bits;
}

// After the tiles: the streams the tile kernel does not write. (i) RAW by the threshold, (ii) RAW by the fallback rule
// (FORMAT.md §8), both expanded from the bitmap block by block (one warp per block); (iii) the empty stream (no tile
// ran). The decision reads the size the plan / the last tile has left in ws.hdr->total_out; *out_total is written
// by one thread (nobody reads it).
template <int W>
__global__ void __launch_bounds__(256) k_bm_finish(EncArgs a) {
    using T = typename IdT<W>::T;
    constexpr unsigned long long E = W / 8;
    pdl_wait();
    pdl_launch_dependents();
    if (a.ws.hdr->ok == 0) return;                                           // (*out_total = 0 since the plan)
    const unsigned long long n = a.ws.hdr->n_ids, body = (n * E + 15ull) & ~15ull, raw_total = 32ull + body;
    const bool raw_thr = n * E < a.thr;
    const unsigned long long have = a.ws.hdr->total_out;                     // raw_thr: = raw_total; n = 0: 48
    const bool first = blockIdx.x == 0 && threadIdx.x == 0;
    if (!raw_thr && have > a.out_cap) {                                      // flagged by the tiles, except when there was none
        if (n == 0 && first) set_status(a.status, BFSC_ERR_DST_TOO_SMALL);
        return;
    }
    const bool to_raw = raw_thr || (a.fallback && have >= raw_total);
    if (!to_raw) {
        if (n == 0 && first) {                                               // (iii) 48 bytes: header, dir[0] = 3
            uint4 h0, h1;
            h0.x = 0x43534642u; h0.y = 1u | ((uint32_t)W << 8) | (a.codec << 16); h0.z = 0; h0.w = 0;
            h1.x = 48u; h1.y = 0; h1.z = 0; h1.w = 0;
            reinterpret_cast<uint4*>(a.out)[0] = h0;
            reinterpret_cast<uint4*>(a.out)[1] = h1;
            reinterpret_cast<uint4*>(a.out)[2] = make_uint4(3u, 0u, 0u, 0u);
            if (a.out_total) *a.out_total = 48ull;
        }
        return;
    }
    if (raw_total > a.out_cap) {
        if (first) { set_status(a.status, BFSC_ERR_DST_TOO_SMALL); if (a.out_total) *a.out_total = 0; }
        return;
    }
    const uint32_t* starts = reinterpret_cast<const uint32_t*>(a.ws.blk_tab);
    const unsigned long long nb_all = (n + kBlk - 1) / kBlk;
    const int lane = threadIdx.x & 31;
    T* y = reinterpret_cast<T*>(a.out + 32);
    if (bm_sparse(a)) {                                                      // the IDs are listed already (k_bm_starts): the RAW body is that list
        const T* list = reinterpret_cast<const T*>(a.list);
        for (unsigned long long j = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; j < n; j += (unsigned long long)gridDim.x * blockDim.x)
            y[j] = list[j];
    } else
    for (unsigned long long g = (unsigned long long)blockIdx.x * 8 + (threadIdx.x >> 5); g < nb_all; g += (unsigned long long)gridDim.x * 8) {
        const uint32_t s = starts[g], e = starts[g + 1];
        if (e <= s) continue;
        const uint32_t w_first = s >> 5, w_last = (e - 1u) >> 5;
        uint32_t rank = 0;
        for (uint32_t w = w_first; w <= w_last && w >= w_first; w += 32) {
            const uint32_t wi = w + (uint32_t)lane;
            uint32_t x = (wi <= w_last && wi >= w) ? a.bitmap[wi] : 0u;
            if (wi == w_first) x &= 0xffffffffu << (s & 31u);
            if (wi == w_last && (e & 31u)) x &= (1u << (e & 31u)) - 1u;
            const uint32_t k = (uint32_t)__popc(x);
            uint32_t inc = k;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) { const uint32_t t = __shfl_up_sync(kFull, inc, o); if (lane >= o) inc += t; }
            uint32_t pos = rank + inc - k;
            rank += __shfl_sync(kFull, inc, 31);
            while (x) {
                const uint32_t b = (uint32_t)__ffs((int)x) - 1u;
                x &= x - 1u;
                y[g * kBlk + pos++] = (T)(a.id_base + 32ull * wi + b);
            }
        }
    }
    for (unsigned long long j = n + (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; j < body / E; j += (unsigned long long)gridDim.x * blockDim.x)
        y[j] = (T)0;                                                         // zero pad
    if (first) {
        uint4 h0, h1;
        h0.x = 0x43534642u; h0.y = 1u | ((uint32_t)W << 8);                  // mode 0
        h0.z = (uint32_t)n; h0.w = (uint32_t)(n >> 32);
        h1.x = (uint32_t)raw_total; h1.y = (uint32_t)(raw_total >> 32); h1.z = 0; h1.w = 0;
        reinterpret_cast<uint4*>(a.out)[0] = h0;
        reinterpret_cast<uint4*>(a.out)[1] = h1;
        if (a.out_total) *a.out_total = raw_total;
    }
}

// Once per device and instantiation: the dynamic shared memory attribute and the resident CTAs per SM.
template <int W, int kSrc>
static int enc_ctas_per_sm(int device) {
    static std::mutex mu;
    static int per_sm[kMaxDevices] = {};
    std::lock_guard<std::mutex> lock(mu);
    if (per_sm[device] == 0) {
        int n = 0;
        if (cudaFuncSetAttribute(k_enc_tiles<W, kSrc>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)EncSmem<W, kSrc>::kBytes) != cudaSuccess)
            return 0;
        if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, k_enc_tiles<W, kSrc>, kEncThreads, EncSmem<W, kSrc>::kBytes) != cudaSuccess || n < 1)
            return 0;
        per_sm[device] = n;
    }
    return per_sm[device];
}

// Once per device: the small-batch kernel's dynamic shared memory and its cluster size. 1 = usable, -1 = this device
// cannot run a cluster of kSmallCtas such CTAs (small batches then take the general path), 0 = a CUDA error.
template <int W>
static int enc_small_init(int device) {
    static std::mutex mu;
    static int state[kMaxDevices] = {};
    std::lock_guard<std::mutex> lock(mu);
    if (state[device] == 0) {
        if (cudaFuncSetAttribute(k_enc_small<W>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SmallSmem<W>::kBytes) != cudaSuccess)
            return 0;
        int n = 0;
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3(kSmallCtas); cfg.blockDim = dim3(kSmallThreads); cfg.dynamicSmemBytes = SmallSmem<W>::kBytes;
        cudaLaunchAttribute at[1];
        at[0].id = cudaLaunchAttributeClusterDimension;
        at[0].val.clusterDim.x = kSmallCtas; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
        cfg.attrs = at; cfg.numAttrs = 1;
        const bool ok = cudaFuncSetAttribute(k_enc_small<W>, cudaFuncAttributeNonPortableClusterSizeAllowed, 1) == cudaSuccess &&
                        cudaOccupancyMaxActiveClusters(&n, k_enc_small<W>, &cfg) == cudaSuccess && n >= 1;
        if (!ok) (void)cudaGetLastError();               // (not an error of the call: the general path runs)
        state[device] = ok ? 1 : -1;
    }
    return state[device];
}

template <int W>
static bfsc_status launch_encode(const EncArgs& a_in, cudaStream_t s) {
    constexpr size_t kSmem = EncSmem<W>::kBytes;
    DeviceInfo dev;
    if (!current_device(&dev)) return BFSC_ERR_CUDA;
    constexpr unsigned long long E = W / 8;
    const bool single = a_in.in_off == nullptr;
    const bool degenerate = single && (a_in.n_single == 0 || a_in.n_single * E < a_in.thr);   // no block: header (+ raw copy) only
    const bool scatter = a_in.dst != nullptr;
    const int per_sm = single ? enc_ctas_per_sm<W, 0>(dev.device) : scatter ? enc_ctas_per_sm<W, 3>(dev.device) : enc_ctas_per_sm<W, 1>(dev.device);
    if (per_sm < 1) return BFSC_ERR_CUDA;
    int grid = dev.sms * per_sm;                                 // one resident wave (every tile is drawn by ticket: any grid size is correct)
    if (single) {
        const unsigned long long n_tiles = ((a_in.n_single + kBlk - 1) / kBlk + kTileR - 1) / kTileR;
        if (!degenerate && n_tiles > a_in.ws.tile_cap) return BFSC_ERR_INVALID_ARG;          // workspace too small
        if (n_tiles < (unsigned long long)grid) grid = n_tiles ? (int)n_tiles : 1;
    }
    int small = 0;
    if (!single && a_in.n_buf <= kSmallMaxBuf && a_in.ws.blk_cap <= kSmallMaxBlocks) {
        small = enc_small_init<W>(dev.device);
        if (small == 0) return BFSC_ERR_CUDA;
    }
    if (small == 1) {
        // a small batch (both bounds known on the host: buffer count, and blocks by the workspace size the caller derived
        // from the total ID count): one launch of one cluster
        EncArgs a = a_in;
        a.grid = kSmallCtas;
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3(kSmallCtas); cfg.blockDim = dim3(kSmallThreads);
        cfg.dynamicSmemBytes = SmallSmem<W>::kBytes; cfg.stream = s;
        cudaLaunchAttribute at[2];
        at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        at[0].val.programmaticStreamSerializationAllowed = 1;
        at[1].id = cudaLaunchAttributeClusterDimension;
        at[1].val.clusterDim.x = kSmallCtas; at[1].val.clusterDim.y = 1; at[1].val.clusterDim.z = 1;
        cfg.attrs = at; cfg.numAttrs = 2;
        BFSC_LAUNCH(cudaLaunchKernelEx(&cfg, k_enc_small<W>, a));
        return BFSC_OK;
    }
    if (!single && (unsigned long long)grid > a_in.ws.tile_cap) grid = (int)a_in.ws.tile_cap;   // (tile_cap >= 2: no more tiles than that)
    EncArgs a = a_in;
    a.grid = (uint32_t)grid;
    const bool fused = !single && a.n_buf <= kFusedMaxBuf;
    if (fused) {                                                 // plan + block table in one launch
        size_t pgrid = (a.ws.blk_cap + 1023) / 1024;
        if (pgrid > (size_t)dev.sms) pgrid = (size_t)dev.sms;
        BFSC_LAUNCH(launch_dep(k_enc_planblocks<W>, pgrid ? (int)pgrid : 1, 1024, 0, s, a));
    } else {
        BFSC_LAUNCH(launch_dep(k_enc_plan<W>, 1, 1024, 0, s, a));
    }
    if (!single && !fused) {
        size_t bgrid = (a.ws.blk_cap + kBlkTabThreads - 1) / kBlkTabThreads;
        if (bgrid > (size_t)dev.sms * 8) bgrid = (size_t)dev.sms * 8;
        BFSC_LAUNCH(launch_dep(k_enc_blocks<W>, bgrid ? (int)bgrid : 1, kBlkTabThreads, 0, s, a));
    }
    if (!degenerate) {
        if (single) BFSC_LAUNCH(launch_dep(k_enc_tiles<W, 0>, grid, kEncThreads, kSmem, s, a));
        else if (scatter) BFSC_LAUNCH(launch_dep(k_enc_tiles<W, 3>, grid, kEncThreads, kSmem, s, a));
        else BFSC_LAUNCH(launch_dep(k_enc_tiles<W, 1>, grid, kEncThreads, kSmem, s, a));
    }
    if (!single || degenerate) {
        uint32_t sgrid = (a.n_buf + 7) / 8;                      // one warp per buffer
        if (sgrid > (uint32_t)dev.sms * 8) sgrid = (uint32_t)dev.sms * 8;
        BFSC_LAUNCH(launch_dep(k_enc_streams<W>, sgrid ? (int)sgrid : 1, 256, 0, s, a));
    }
    if (single && a.fallback) {
        size_t fgrid = (a.n_single * E / (256 * 16 * 4)) + 1;    // 16 bytes per thread and round, a few rounds
        if (fgrid > (size_t)dev.sms * 8) fgrid = (size_t)dev.sms * 8;
        BFSC_LAUNCH(launch_dep(k_enc_fallback<W>, (int)fgrid, 256, 0, s, a));
    }
    return BFSC_OK;
}

// bfsc_compress_bitmap: count -> plan -> starts -> tiles -> finish (the tile count is known on the device only: one
// resident wave of CTAs, or fewer when even a full bitmap has fewer tiles; tiles are drawn by ticket).
template <int W>
static bfsc_status launch_encode_bitmap(const EncArgs& a_in, cudaStream_t s) {
    constexpr size_t kSmem = EncSmem<W, 2>::kBytes;
    DeviceInfo dev;
    if (!current_device(&dev)) return BFSC_ERR_CUDA;
    const int per_sm = enc_ctas_per_sm<W, 2>(dev.device);
    if (per_sm < 1) return BFSC_ERR_CUDA;
    EncArgs a = a_in;
    int grid = dev.sms * per_sm;
    const unsigned long long max_tiles = ((a.n_bits + kBlk - 1) / kBlk + kTileR - 1) / kTileR;
    if (max_tiles > a.ws.tile_cap) return BFSC_ERR_INVALID_ARG;              // workspace too small
    if (max_tiles < (unsigned long long)grid) grid = max_tiles ? (int)max_tiles : 1;
    a.grid = (uint32_t)grid;
    size_t cgrid = (size_t)((a.n_chunks + 7) / 8), sgrid = (size_t)((a.n_super + 7) / 8);
    if (cgrid > (size_t)dev.sms * 8) cgrid = (size_t)dev.sms * 8;
    sgrid = (size_t)a.n_super;                                       // k_bm_count: a CTA takes a super-chunk
    if (sgrid > (size_t)dev.sms * 8) sgrid = (size_t)dev.sms * 8;
    if (cgrid < 1) cgrid = 1;
    if (sgrid < 1) sgrid = 1;
    BFSC_LAUNCH(launch_dep(k_bm_count, (int)sgrid, 256, 0, s, a));
    BFSC_LAUNCH(launch_dep(k_bm_plan<W>, 1, 1024, 0, s, a));
    size_t tgrid = (size_t)((a.n_chunks + 8 * kStartsPer - 1) / (8 * kStartsPer));
    if (tgrid > (size_t)dev.sms * 8) tgrid = (size_t)dev.sms * 8;
    if (tgrid < 1) tgrid = 1;
    BFSC_LAUNCH(launch_dep(k_bm_starts<W>, (int)tgrid, 256, 0, s, a));
    BFSC_LAUNCH(launch_dep(k_enc_tiles<W, 2>, grid, kEncThreads, kSmem, s, a));
    if (a.thr > 0 || a.fallback)                                     // (else no stream can end up RAW, and the plan wrote the empty one)
        BFSC_LAUNCH(launch_dep(k_bm_finish<W>, (int)cgrid, 256, 0, s, a));
    return BFSC_OK;
}

static bfsc_status encode_common(bfsc_codec codec, const void* d_ids, const uint64_t* d_in_off, size_t n_single, size_t n_buf,
                                 bfsc_dtype t, size_t thr, void* d_out, size_t out_cap, uint64_t* d_out_off,
                                 uint64_t* d_out_total, void* ws, size_t ws_bytes, uint32_t* d_status, void* stream,
                                 void* const* d_dst = nullptr, uint64_t* d_out_sizes = nullptr) {
    if (t != BFSC_U32 && t != BFSC_U64) return BFSC_ERR_INVALID_ARG;
    const uint32_t exclusive = ((uint32_t)codec & (uint32_t)BFSC_CODEC_FLAG_EXCLUSIVE) ? 1u : 0u;
    const uint32_t fallback = ((uint32_t)codec & (uint32_t)BFSC_CODEC_FLAG_RAW_FALLBACK) ? 1u : 0u;
    codec = (bfsc_codec)((uint32_t)codec & ~(uint32_t)(BFSC_CODEC_FLAG_EXCLUSIVE | BFSC_CODEC_FLAG_RAW_FALLBACK));
    if (codec != BFSC_CODEC_PFOR && codec != BFSC_CODEC_BP128) return BFSC_ERR_INVALID_ARG;
    if (fallback && d_in_off) return BFSC_ERR_UNSUPPORTED;                  // FORMAT.md §8: single-buffer calls
    if ((!d_out && !d_dst) || !ws || n_buf > 0x7fffffffu) return BFSC_ERR_INVALID_ARG;
    if (d_dst && (d_out || !d_in_off || !d_out_sizes)) return BFSC_ERR_INVALID_ARG;     // scatter: batch calls, no common output
    if (((uintptr_t)d_ids & 15) || ((uintptr_t)d_out & 15) || ((uintptr_t)ws & 15)) return BFSC_ERR_INVALID_ARG;
    if (!d_ids && (d_in_off || n_single)) return BFSC_ERR_INVALID_ARG;
    EncArgs a = {};
    if (!ws_carve(ws, ws_bytes, n_buf, &a.ws)) return BFSC_ERR_INVALID_ARG;
    a.fallback = fallback;
    a.ids = d_ids; a.in_off = (const unsigned long long*)d_in_off; a.n_single = n_single;
    a.n_buf = (uint32_t)n_buf; a.codec = (uint32_t)codec; a.exclusive = exclusive; a.grid = 0; a.thr = thr; a.out = (unsigned char*)d_out; a.out_cap = out_cap;
    a.out_off = (unsigned long long*)d_out_off; a.out_total = (unsigned long long*)d_out_total; a.status = d_status;
    if (d_dst) {                                         // out == nullptr: offsets into it are addresses
        a.dst = reinterpret_cast<const unsigned long long*>(d_dst); a.dst_cap = out_cap; a.out_cap = ~0ull;
        a.out_sizes = (unsigned long long*)d_out_sizes;
    }
    return t == BFSC_U32 ? launch_encode<32>(a, (cudaStream_t)stream) : launch_encode<64>(a, (cudaStream_t)stream);
}

}  // namespace bfsc

#ifdef BFSC_CHECKED
extern "C" void bfsc_debug_checks_encode(unsigned int* h_failures_and_line) {      // BFSC_CHECK violations of the encode kernels so far
    cudaDeviceSynchronize();
    cudaMemcpyFromSymbol(h_failures_and_line, bfsc::g_bfsc_check, 2 * sizeof(unsigned int));
}
namespace bfsc {
__global__ void k_check_selftest() { BFSC_CHECK(threadIdx.x != 3); }               // one violation, on purpose
}
// Proves that a violated BFSC_CHECK is seen: runs one, returns what the counters then say in h_seen[0..1] (failures added,
// line recorded), and puts the counters back as they were.
extern "C" void bfsc_debug_check_selftest(unsigned int* h_seen) {
    unsigned int before[2], after[2];
    cudaDeviceSynchronize();
    cudaMemcpyFromSymbol(before, bfsc::g_bfsc_check, sizeof(before));
    const unsigned int zero[2] = {0u, 0u};
    cudaMemcpyToSymbol(bfsc::g_bfsc_check, zero, sizeof(zero));
    bfsc::k_check_selftest<<<1, 32>>>();
    cudaDeviceSynchronize();
    cudaMemcpyFromSymbol(after, bfsc::g_bfsc_check, sizeof(after));
    cudaMemcpyToSymbol(bfsc::g_bfsc_check, before, sizeof(before));
    h_seen[0] = after[0]; h_seen[1] = after[1];
}
#endif

extern "C" bfsc_status bfsc_compress_codec(bfsc_codec codec, const void* d_ids, size_t n_ids, bfsc_dtype t,
                                           size_t raw_threshold_bytes, void* d_out, size_t out_capacity,
                                           uint64_t* d_out_bytes, void* d_workspace, size_t workspace_bytes,
                                           uint32_t* d_status, void* cuda_stream) {
    if (!d_out_bytes) return BFSC_ERR_INVALID_ARG;
    return bfsc::encode_common(codec, d_ids, nullptr, n_ids, 1, t, raw_threshold_bytes, d_out, out_capacity, nullptr,
                               d_out_bytes, d_workspace, workspace_bytes, d_status, cuda_stream);
}

extern "C" bfsc_status bfsc_compress_bitmap(bfsc_codec codec, const uint32_t* d_bitmap, size_t n_bits, uint64_t id_base,
                                            bfsc_dtype t, size_t raw_threshold_bytes, void* d_out, size_t out_capacity,
                                            uint64_t* d_out_bytes, void* d_workspace, size_t workspace_bytes,
                                            uint32_t* d_status, void* cuda_stream) {
    using namespace bfsc;
    if (t != BFSC_U32 && t != BFSC_U64) return BFSC_ERR_INVALID_ARG;
    const uint32_t fallback = ((uint32_t)codec & (uint32_t)BFSC_CODEC_FLAG_RAW_FALLBACK) ? 1u : 0u;
    codec = (bfsc_codec)((uint32_t)codec & ~(uint32_t)(BFSC_CODEC_FLAG_EXCLUSIVE | BFSC_CODEC_FLAG_RAW_FALLBACK));   // (exclusive: no effect here)
    if (codec != BFSC_CODEC_PFOR && codec != BFSC_CODEC_BP128) return BFSC_ERR_INVALID_ARG;
    if (!d_out || !d_out_bytes || !d_workspace || (n_bits && !d_bitmap)) return BFSC_ERR_INVALID_ARG;
    if ((unsigned long long)n_bits >= (1ull << 32)) return BFSC_ERR_INVALID_ARG;
    if (((uintptr_t)d_bitmap & 15) || ((uintptr_t)d_out & 15) || ((uintptr_t)d_workspace & 15)) return BFSC_ERR_INVALID_ARG;
    const size_t std_bytes = align_up(ws_bytes_for(n_bits, 1), 16), n_chunks = (n_bits + kChunkBits - 1) / kChunkBits;
    const size_t n_super = (n_chunks + kSuperChunks - 1) / kSuperChunks;
    if (workspace_bytes < std_bytes + bitmap_extra_ws_bytes(n_bits)) return BFSC_ERR_INVALID_ARG;
    EncArgs a = {};
    if (!ws_carve(d_workspace, std_bytes, 1, &a.ws)) return BFSC_ERR_INVALID_ARG;
    a.bitmap = d_bitmap; a.n_bits = n_bits; a.id_base = id_base;
    a.chunk = reinterpret_cast<uint32_t*>(static_cast<char*>(d_workspace) + std_bytes);       // 16-byte aligned: read as uint4
    a.super = reinterpret_cast<unsigned long long*>(a.chunk + n_super * kSuperChunks);
    a.list = static_cast<char*>(d_workspace) + std_bytes + align_up(8 * (n_super + 1) + 4 * 32 * n_super + 16, 16);
    a.n_chunks = n_chunks; a.n_super = n_super;
    a.fallback = fallback; a.n_buf = 1; a.codec = (uint32_t)codec; a.thr = raw_threshold_bytes;
    a.out = (unsigned char*)d_out; a.out_cap = out_capacity; a.out_total = (unsigned long long*)d_out_bytes; a.status = d_status;
    return t == BFSC_U32 ? launch_encode_bitmap<32>(a, (cudaStream_t)cuda_stream) : launch_encode_bitmap<64>(a, (cudaStream_t)cuda_stream);
}

// ---- FORMAT.md §10: a (visited) bitmap as a container that lists its MINORITY bits, or holds the bitmap itself.
// count -> select (the bitmap or its complement, tail bits cleared, into the workspace) -> the bitmap encode chain above on
// that copy, its stream straight behind the container header, capped at the size of the bitmap itself (a stream that does
// not fit is not smaller either) -> finish (header; the raw bitmap over the stream if that did not pay).
namespace bfsc {
struct VbScratch { unsigned long long count, stream_bytes, n_decoded, n_listed; unsigned int status, kind, skip, pad; };
static_assert(sizeof(VbScratch) <= 256, "VbScratch");

__device__ __forceinline__ uint32_t vb_word(const uint32_t* __restrict__ bm, unsigned long long w, unsigned long long n_bits, bool invert) {
    const unsigned long long bit0 = 32ull * w;
    if (bit0 >= n_bits) return 0u;
    uint32_t x = bm[w];
    if (invert) x = ~x;
    if (n_bits - bit0 < 32) x &= (1u << (uint32_t)(n_bits - bit0)) - 1u;
    return x;
}
// (every kernel of the container is launched like the others of the library: programmatic dependent launch, no memset node)
__global__ void __launch_bounds__(256) k_vb_count(const uint32_t* __restrict__ bm, unsigned long long n_bits, unsigned long long* __restrict__ partial) {
    __shared__ unsigned long long s_c[8];
    pdl_wait();                                                      // the call before this one is complete (workspace)
    pdl_launch_dependents();
    const unsigned long long words = (n_bits + 31) / 32;
    unsigned long long c = 0;
    for (unsigned long long w = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; w < words; w += (unsigned long long)gridDim.x * blockDim.x)
        c += (unsigned long long)__popc(vb_word(bm, w, n_bits, false));
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) c += __shfl_xor_sync(kFull, c, o);
    if ((threadIdx.x & 31) == 0) s_c[threadIdx.x >> 5] = c;
    __syncthreads();
    if (threadIdx.x == 0) partial[blockIdx.x] = s_c[0] + s_c[1] + s_c[2] + s_c[3] + s_c[4] + s_c[5] + s_c[6] + s_c[7];   // one sum per CTA
}
__global__ void __launch_bounds__(256) k_vb_select(const uint32_t* __restrict__ bm, unsigned long long n_bits, uint32_t* __restrict__ wb,
                                                   unsigned long long wb_words, VbScratch* sc, const unsigned long long* __restrict__ partial, int n_partial) {
    __shared__ unsigned long long s_c[8];
    pdl_wait();
    pdl_launch_dependents();
    unsigned long long c = 0;                                        // every CTA adds up the per-CTA popcounts for itself
    for (int i = threadIdx.x; i < n_partial; i += blockDim.x) c += partial[i];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) c += __shfl_xor_sync(kFull, c, o);
    if ((threadIdx.x & 31) == 0) s_c[threadIdx.x >> 5] = c;
    __syncthreads();
    const unsigned long long count = s_c[0] + s_c[1] + s_c[2] + s_c[3] + s_c[4] + s_c[5] + s_c[6] + s_c[7];
    if (blockIdx.x == 0 && threadIdx.x == 0) { sc->count = count; sc->stream_bytes = 0; sc->status = 0; }
    const bool invert = count > n_bits - count;                      // the clear bits are the minority
    for (unsigned long long w = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; w < wb_words; w += (unsigned long long)gridDim.x * blockDim.x)
        wb[w] = vb_word(bm, w, n_bits, invert);
}
__global__ void __launch_bounds__(256) k_vb_finish(const uint32_t* __restrict__ bm, unsigned long long n_bits, unsigned char* __restrict__ out,
                                                   unsigned long long raw_bytes, const VbScratch* sc, unsigned long long* out_bytes) {
    pdl_wait();
    pdl_launch_dependents();
    const unsigned long long k = sc->count, sb = sc->stream_bytes;
    const bool invert = k > n_bits - k;
    const uint32_t kind = (sc->status == 0u && sb != 0ull && sb < raw_bytes) ? (invert ? 2u : 1u) : 0u;
    if (kind == 0u) {                                                // the bitmap itself (tail bits cleared, zero pad)
        uint32_t* y = reinterpret_cast<uint32_t*>(out + 32);
        for (unsigned long long w = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; w < raw_bytes / 4; w += (unsigned long long)gridDim.x * blockDim.x)
            y[w] = vb_word(bm, w, n_bits, false);
    }
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        const unsigned long long total = 32ull + (kind ? sb : raw_bytes), n_listed = kind ? (invert ? n_bits - k : k) : 0ull;
        uint4 h0, h1;
        h0.x = 0x56534642u;                                          // "BFSV"
        h0.y = 1u | (32u << 8) | (kind << 16);
        h0.z = (uint32_t)n_bits; h0.w = (uint32_t)(n_bits >> 32);
        h1.x = (uint32_t)total; h1.y = (uint32_t)(total >> 32);
        h1.z = (uint32_t)n_listed; h1.w = (uint32_t)(n_listed >> 32);
        reinterpret_cast<uint4*>(out)[0] = h0;
        reinterpret_cast<uint4*>(out)[1] = h1;
        *out_bytes = total;
    }
}
}  // namespace bfsc

extern "C" size_t bfsc_vbitmap_bound(size_t n_bits) { return 32 + bfsc::align_up(4 * ((n_bits + 31) / 32), 16); }
extern "C" size_t bfsc_vbitmap_workspace_bytes(size_t n_bits) {
    return 256 + bfsc::align_up(4 * ((n_bits + 31) / 32) + 16, 256) + bfsc_bitmap_workspace_bytes(n_bits, BFSC_U32);
}

extern "C" bfsc_status bfsc_compress_vbitmap(bfsc_codec codec, const uint32_t* d_bitmap, size_t n_bits, void* d_out,
                                             size_t out_capacity, uint64_t* d_out_bytes, void* d_workspace,
                                             size_t workspace_bytes, uint32_t* d_status, void* cuda_stream) {
    using namespace bfsc;
    codec = (bfsc_codec)((uint32_t)codec & ~(uint32_t)BFSC_CODEC_FLAG_EXCLUSIVE);
    if (codec != BFSC_CODEC_PFOR && codec != BFSC_CODEC_BP128) return BFSC_ERR_INVALID_ARG;
    if (!d_out || !d_out_bytes || !d_workspace || (n_bits && !d_bitmap) || (unsigned long long)n_bits > (1ull << 32)) return BFSC_ERR_INVALID_ARG;
    if (((uintptr_t)d_out & 15) || ((uintptr_t)d_workspace & 15) || ((uintptr_t)d_bitmap & 3)) return BFSC_ERR_INVALID_ARG;
    if (workspace_bytes < bfsc_vbitmap_workspace_bytes(n_bits)) return BFSC_ERR_INVALID_ARG;
    if (out_capacity < bfsc_vbitmap_bound(n_bits)) return BFSC_ERR_DST_TOO_SMALL;
    (void)d_status;                                                  // (nothing can go wrong on the device that is not an argument error above)
    cudaStream_t s = (cudaStream_t)cuda_stream;
    DeviceInfo dev;
    if (!current_device(&dev)) return BFSC_ERR_CUDA;
    const size_t words = (n_bits + 31) / 32, raw_bytes = align_up(4 * words, 16), wb_bytes = align_up(4 * words + 16, 256);
    VbScratch* sc = reinterpret_cast<VbScratch*>(d_workspace);
    uint32_t* wb = reinterpret_cast<uint32_t*>(static_cast<char*>(d_workspace) + 256);
    void* ws_bm = static_cast<char*>(d_workspace) + 256 + wb_bytes;
    int grid = (int)((words + 255) / 256);
    if (grid > dev.sms * 8) grid = dev.sms * 8;
    if (grid < 1) grid = 1;
    // per-CTA popcounts: at the start of the bitmap-encode workspace, which nothing uses before k_vb_select has read them
    unsigned long long* partial = reinterpret_cast<unsigned long long*>(ws_bm);
    if ((size_t)grid * 8 > workspace_bytes - 256 - wb_bytes) return BFSC_ERR_INVALID_ARG;
    BFSC_LAUNCH(launch_dep_v(k_vb_count, grid, 256, 0, s, d_bitmap, (unsigned long long)n_bits, partial));
    BFSC_LAUNCH(launch_dep_v(k_vb_select, grid, 256, 0, s, d_bitmap, (unsigned long long)n_bits, wb, (unsigned long long)(wb_bytes / 4), sc,
                           (const unsigned long long*)partial, grid));      // (every word of the copy: the encode kernels read whole 16-byte chunks)
    const bfsc_status rc = bfsc_compress_bitmap(codec, wb, n_bits, 0, BFSC_U32, 0, static_cast<unsigned char*>(d_out) + 32, raw_bytes,
                                                reinterpret_cast<uint64_t*>(&sc->stream_bytes), ws_bm, workspace_bytes - 256 - wb_bytes, &sc->status, cuda_stream);
    if (rc != BFSC_OK) return rc;
    BFSC_LAUNCH(launch_dep_v(k_vb_finish, grid, 256, 0, s, d_bitmap, (unsigned long long)n_bits, static_cast<unsigned char*>(d_out),
                           (unsigned long long)raw_bytes, (const VbScratch*)sc, (unsigned long long*)d_out_bytes));
    return BFSC_OK;
}

extern "C" bfsc_status bfsc_compress(const void* d_ids, size_t n_ids, bfsc_dtype t, size_t raw_threshold_bytes,
                                     void* d_out, size_t out_capacity, uint64_t* d_out_bytes, void* d_workspace,
                                     size_t workspace_bytes, uint32_t* d_status, void* cuda_stream) {
    return bfsc_compress_codec(BFSC_CODEC_PFOR, d_ids, n_ids, t, raw_threshold_bytes, d_out, out_capacity, d_out_bytes,
                               d_workspace, workspace_bytes, d_status, cuda_stream);
}

// ---- bfsc_compress_noalloc (include/bfsc.h): the workspace of a single-buffer call of up to BFSC_NOALLOC_MAX_IDS IDs
// lives in the library image. In HOST code the array's name is a host-side stand-in, not a device address: the address
// the kernels get comes from cudaGetSymbolAddress, once per device, with that device current.
namespace bfsc {
static __device__ __align__(256) unsigned char g_noalloc_scratch[BFSC_NOALLOC_SCRATCH_BYTES];

static void* noalloc_scratch(int device) {               // device address of the array on `device` (the current one), or nullptr
    static std::mutex mu;
    static void* addr[kMaxDevices] = {};
    std::lock_guard<std::mutex> lock(mu);
    if (addr[device] == nullptr) {
        void* p = nullptr;
        if (cudaGetSymbolAddress(&p, g_noalloc_scratch) != cudaSuccess || p == nullptr) return nullptr;
        addr[device] = p;
    }
    return addr[device];
}
}  // namespace bfsc

extern "C" bfsc_status bfsc_compress_noalloc(const void* d_ids, size_t n_ids, bfsc_dtype t, size_t raw_threshold_bytes,
                                             void* d_out, size_t out_capacity, uint64_t* d_out_bytes,
                                             uint32_t* d_status, void* cuda_stream) {
    using namespace bfsc;
    if (!d_out_bytes) return BFSC_ERR_INVALID_ARG;
    if (n_ids > BFSC_NOALLOC_MAX_IDS) return BFSC_ERR_INVALID_ARG;       // beyond what the built-in scratch array holds
    static_assert(BFSC_NOALLOC_SCRATCH_BYTES % 256 == 0, "scratch size");
    if (ws_bytes_for(BFSC_NOALLOC_MAX_IDS, 1) > BFSC_NOALLOC_SCRATCH_BYTES) return BFSC_ERR_INVALID_ARG;   // (a build-time property)
    DeviceInfo dev;
    if (!current_device(&dev)) return BFSC_ERR_CUDA;
    void* ws = noalloc_scratch(dev.device);
    if (ws == nullptr) return BFSC_ERR_CUDA;
    return encode_common(BFSC_CODEC_PFOR, d_ids, nullptr, n_ids, 1, t, raw_threshold_bytes, d_out, out_capacity, nullptr,
                         d_out_bytes, ws, BFSC_NOALLOC_SCRATCH_BYTES, d_status, cuda_stream);
}

extern "C" bfsc_status bfsc_compress_batch_codec(bfsc_codec codec, const void* d_ids, const uint64_t* d_in_offsets,
                                                 size_t n_buf, bfsc_dtype t, size_t raw_threshold_bytes, void* d_out,
                                                 size_t out_capacity, uint64_t* d_out_offsets, void* d_workspace,
                                                 size_t workspace_bytes, uint32_t* d_status, void* cuda_stream) {
    if (!d_in_offsets || !d_out_offsets) return BFSC_ERR_INVALID_ARG;
    return bfsc::encode_common(codec, d_ids, d_in_offsets, 0, n_buf, t, raw_threshold_bytes, d_out, out_capacity,
                               d_out_offsets, nullptr, d_workspace, workspace_bytes, d_status, cuda_stream);
}

extern "C" bfsc_status bfsc_compress_batch(const void* d_ids, const uint64_t* d_in_offsets, size_t n_buf,
                                           bfsc_dtype t, size_t raw_threshold_bytes, void* d_out,
                                           size_t out_capacity, uint64_t* d_out_offsets, void* d_workspace,
                                           size_t workspace_bytes, uint32_t* d_status, void* cuda_stream) {
    return bfsc_compress_batch_codec(BFSC_CODEC_PFOR, d_ids, d_in_offsets, n_buf, t, raw_threshold_bytes, d_out,
                                     out_capacity, d_out_offsets, d_workspace, workspace_bytes, d_status, cuda_stream);
}

extern "C" bfsc_status bfsc_compress_batch_scatter(bfsc_codec codec, const void* d_ids, const uint64_t* d_in_offsets,
                                                   size_t n_buf, bfsc_dtype t, size_t raw_threshold_bytes,
                                                   void* const* d_dst, size_t dst_capacity, uint64_t* d_out_bytes,
                                                   void* d_workspace, size_t workspace_bytes, uint32_t* d_status,
                                                   void* cuda_stream) {
    if (!d_in_offsets || !d_dst || !d_out_bytes) return BFSC_ERR_INVALID_ARG;
    return bfsc::encode_common(codec, d_ids, d_in_offsets, 0, n_buf, t, raw_threshold_bytes, nullptr, dst_capacity,
                               nullptr, nullptr, d_workspace, workspace_bytes, d_status, cuda_stream, d_dst, d_out_bytes);
}
