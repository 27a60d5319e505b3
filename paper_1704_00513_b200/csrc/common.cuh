// common.cuh — shared device/host helpers of the bfsc CUDA library (sm_100a only).
// Product code: shares nothing with oracle/. Layout per FORMAT.md v1.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/bfsc.h"

namespace bfsc {

constexpr int kBlk = 128;               // IDs per block
constexpr int kWarp = 32;
constexpr uint32_t kFull = 0xffffffffu;

template <int W> struct IdT;
template <> struct IdT<32> { using T = uint32_t; };
template <> struct IdT<64> { using T = uint64_t; };

// ---- workspace layout (device) -------------------------------------------------------
// [WsHeader 256 B][blk_first u64 (n_buf+1)][fixed_prefix u64 (n_buf+1)][stream_start u64 (n_buf+1)]
// [tile_state: tile_cap entries of kStateStride u64 (one 64-byte entry per tile: the look-back polls
//  of the tiles in flight then spread over many L2 slices instead of a few hot lines)]
// [blk_tab: blk_cap entries of 32 B — batch calls: where each block of the batch lives (EncBlk / DecBlk),
//  written by k_*_blocks after the plan, so that the tile kernels find a block with ONE load]
struct WsHeader {
    unsigned long long total_blocks;    // blocks of all PFOR streams of the batch
    unsigned long long fixed_total;     // sum of per-stream fixed bytes (header+directory | header+raw)
    unsigned long long total_out;       // encode: total output bytes; decode: total ids
    unsigned int ok;                    // 1 = plan valid and capacity sufficient
    unsigned int ticket;                // tile ticket counter (fused encode)
    unsigned long long grand16;         // encode: sum of all block sizes in 16-B units (written by the last tile)
    unsigned long long n_ids;           // bfsc_compress_bitmap: set bits of the bitmap = IDs of the stream (k_bm_plan)
    unsigned long long pad[26];
};
static_assert(sizeof(WsHeader) == 256, "WsHeader");

struct WsView {
    WsHeader* hdr;
    unsigned long long* blk_first;      // n_buf+1 : first global block of each buffer
    unsigned long long* fixed_prefix;   // n_buf+1 : exclusive prefix of fixed bytes (decode: of IDs)
    unsigned long long* stream_start;   // n_buf+1 : encode: 1 + byte offset of the stream (0 = not yet known)
    unsigned long long* tile_state;     // tile_cap * kStateStride
    uint4* blk_tab;                     // blk_cap * 2 (32 B per block), batch calls only
    size_t blk_cap;
    size_t tile_cap;
};

constexpr int kTileBlocks = 64;         // blocks per encode tile (8 worker warps x 8 blocks)
constexpr int kStateStride = 8;         // u64 words between look-back states (64 B)
constexpr size_t kTileWsBytes = 8 * kStateStride + 32 * kTileBlocks;   // workspace per tile: state + block table

// Block table entries (batch calls). Encode: where the block's IDs are. Decode: where its stream is, which
// block of the stream it is and where its IDs go.
struct EncBlk { unsigned long long xoff; uint32_t m; uint32_t buf; uint4 pad; };              // first ID (element), valid IDs, buffer
struct DecBlk { unsigned long long s_begin, x_index; uint32_t k, m, total16, nb; };           // stream start (byte), first ID (element), block, valid IDs, stream bytes / 16, blocks of the stream
static_assert(sizeof(EncBlk) == 32 && sizeof(DecBlk) == 32, "block table entries are 32 B");

__host__ __device__ inline size_t align_up(size_t x, size_t k) { return (x + k - 1) / k * k; }

__host__ inline size_t ws_bytes_for(size_t n_ids_total, size_t n_buf) {
    const size_t blk_cap = n_ids_total / kBlk + n_buf + 1;
    const size_t tile_cap = blk_cap / kTileBlocks + 2;
    return sizeof(WsHeader) + 3 * align_up(8 * (n_buf + 1), 16) + kTileWsBytes * tile_cap + 256;
}

// bfsc_compress_bitmap: behind the standard workspace of one stream of n_bits IDs — the set bits before every super-chunk of
// 32 x 1024 bits (u64, + the total) and, inside its super-chunk, before every chunk (u32)
__host__ inline size_t bitmap_list_ids(size_t n_bits) { return n_bits / 16 + 128; }      // IDs the sparse path's list holds (used up to one set bit in 16)
__host__ inline size_t bitmap_extra_ws_bytes(size_t n_bits) {
    const size_t n_super = (n_bits + 32767) / 32768;
    return align_up(8 * (n_super + 1) + 4 * 32 * n_super + 16, 16) + 8 * bitmap_list_ids(n_bits);   // (the list: 8 bytes per ID, either width)
}

// Carves the workspace; the capacities are derived from the bytes actually provided.
__host__ inline bool ws_carve(void* ws, size_t bytes, size_t n_buf, WsView* v) {
    const size_t fixed = sizeof(WsHeader) + 3 * align_up(8 * (n_buf + 1), 16);
    if (bytes < fixed + kTileWsBytes * 2) return false;
    const size_t tile_cap = (bytes - fixed) / kTileWsBytes;
    char* p = (char*)ws;
    v->hdr = (WsHeader*)p; p += sizeof(WsHeader);
    v->blk_first = (unsigned long long*)p; p += align_up(8 * (n_buf + 1), 16);
    v->fixed_prefix = (unsigned long long*)p; p += align_up(8 * (n_buf + 1), 16);
    v->stream_start = (unsigned long long*)p; p += align_up(8 * (n_buf + 1), 16);
    v->tile_state = (unsigned long long*)p; p += 8 * kStateStride * tile_cap;
    v->blk_tab = (uint4*)p;
    v->tile_cap = tile_cap;
    v->blk_cap = (tile_cap - 1) * kTileBlocks;
    return true;
}

// ---- -DBFSC_CHECKED (python -m paper_1704_00513_b200.build --checked, or BFSC_CHECKED=1 in the environment of the tests):
// every BFSC_CHECK in the kernels is evaluated — shared-memory slot indices, global stores against out_capacity /
// ids_capacity / the bitmap — and a violation is counted (first failing source line kept) instead of trapping, so that a
// whole test run can be made under it and asked for the count at the end (bfsc_debug_checks_encode / _decode; one
// counter per translation unit). The normal build compiles the checks away. compute-sanitizer is not available on
// the GPU pool this library is developed on; this is its stand-in.
#ifdef BFSC_CHECKED
static __device__ unsigned int g_bfsc_check[2];          // failures, first failing line
#define BFSC_CHECK(cond)                                                                     \
    do {                                                                                     \
        if (!(cond)) { atomicAdd(&g_bfsc_check[0], 1u); atomicCAS(&g_bfsc_check[1], 0u, (unsigned)__LINE__); } \
    } while (0)
#else
#define BFSC_CHECK(cond) do { } while (0)
#endif

// ---- device helpers ------------------------------------------------------------------
__device__ __forceinline__ void set_status(uint32_t* st, uint32_t code) {
    if (st) atomicCAS(st, 0u, code);
}

__device__ __forceinline__ int lane_id() { return threadIdx.x & 31; }

// PTX shl/shr clamp shift amounts >= 32 (result 0); C++ << would be undefined there.
__device__ __forceinline__ uint32_t shl32(uint32_t x, uint32_t s) {
    uint32_t r; asm("shl.b32 %0, %1, %2;" : "=r"(r) : "r"(x), "r"(s)); return r;
}
__device__ __forceinline__ uint32_t shr32(uint32_t x, uint32_t s) {
    uint32_t r; asm("shr.u32 %0, %1, %2;" : "=r"(r) : "r"(x), "r"(s)); return r;
}
__device__ __forceinline__ uint64_t shl64(uint64_t x, uint32_t s) {
    uint64_t r; asm("shl.b64 %0, %1, %2;" : "=l"(r) : "l"(x), "r"(s)); return r;
}
__device__ __forceinline__ uint64_t shr64(uint64_t x, uint32_t s) {
    uint64_t r; asm("shr.u64 %0, %1, %2;" : "=l"(r) : "l"(x), "r"(s)); return r;
}
__device__ __forceinline__ int width32(uint32_t v) { return 32 - __clz(v); }
__device__ __forceinline__ int width64(uint64_t v) { return 64 - __clzll(v); }

// bytes of the exception area: n ? align16(align_{W/8}(n) + n*W/8) : 0      (FORMAT.md §2)
template <int W>
__device__ __forceinline__ uint32_t exc_bytes(uint32_t n) {
    constexpr uint32_t E = W / 8;
    uint32_t a = ((n + E - 1) & ~(E - 1)) + n * E;
    return n ? ((a + 15u) & ~15u) : 0u;
}

// Decoding into a frontier bitmap (FORMAT.md §9): bit (x - id_base) of bm for every decoded ID x. bm == nullptr: IDs go to
// the ID array as usual.
struct BitSink { uint32_t* bm; unsigned long long id_base, n_bits; uint32_t* status; uint32_t* visited; };
// Up to four (word, mask) pairs into the sink: plain ORs into the bitmap, or (bfsc_decompress_to_frontier, Algorithm 4
// lines 11-13) ORs into the visited bitmap first — what was not visited before goes into the frontier bitmap. The
// atomic's return value says which of the bits were visited before (exactly once per vertex, whoever else updates the
// same word); it costs a round trip to L2, so the (up to four) visited updates of a call go out TOGETHER and their
// results are looked at afterwards (sparse levels: 28 -> 26 us per call on 8 x 4096 IDs over 2^16-2^20 vertices; what
// remains is the rate at which one warp's scattered atomics are accepted, 32 addresses per instruction: with the same
// IDs packed 4 to a word the call takes 11 us). Measured alternative to the returning atomic: a plain load
// of the visited word + a non-returning atomic — no faster (the atomics of the same SM keep invalidating the L1 lines
// the loads would hit: 59.6 against 54.1 us on the 2^25-bit frontier of bench.py).
template <int N>
__device__ __forceinline__ void sink_or_n(const BitSink& s, const uint32_t (&w)[N], const uint32_t (&mk)[N]) {
    if (s.visited != nullptr) {
        uint32_t old[N];
#pragma unroll
        for (int c = 0; c < N; c++) {
            BFSC_CHECK(mk[c] == 0u || (unsigned long long)w[c] < (s.n_bits + 31) / 32);
            old[c] = mk[c] ? atomicOr(s.visited + w[c], mk[c]) : 0xffffffffu;
        }
#pragma unroll
        for (int c = 0; c < N; c++) {
            const uint32_t fresh = mk[c] & ~old[c];
            if (fresh) atomicOr(s.bm + w[c], fresh);
        }
    } else {
#pragma unroll
        for (int c = 0; c < N; c++) {
            BFSC_CHECK(mk[c] == 0u || (unsigned long long)w[c] < (s.n_bits + 31) / 32);
            if (mk[c]) atomicOr(s.bm + w[c], mk[c]);
        }
    }
}
// Four consecutive decoded IDs (the first nvalid of them count). Neighbours that fall into the same 32-bit word go
// out as ONE atomic OR (sorted dense frontiers: usually all four). An ID outside the bitmap: DST_TOO_SMALL, not set.
template <typename T>
__device__ __forceinline__ void set_bits4(const BitSink& s, T v0, T v1, T v2, T v3, int nvalid) {
    const T v[4] = {v0, v1, v2, v3};
    {   // Usual case (a sorted, dense frontier): all four count, all lie inside the bitmap, in the word of the first one or
        // the word after it: one range test for the four, one or two atomics. Anything else takes the general path below.
        const T r0 = (T)(v0 - (T)s.id_base), r1 = (T)(v1 - (T)s.id_base), r2 = (T)(v2 - (T)s.id_base), r3 = (T)(v3 - (T)s.id_base);
        if (nvalid >= 4 && (unsigned long long)(r0 | r1 | r2 | r3) < s.n_bits) {       // (the OR is >= each of them)
            const uint32_t q0 = (uint32_t)r0, w0 = q0 >> 5;                            // n_bits <= 2^32: the offsets fit 32 bits
            const uint32_t d1 = ((uint32_t)r1 >> 5) - w0, d2 = ((uint32_t)r2 >> 5) - w0, d3 = ((uint32_t)r3 >> 5) - w0;
            if ((d1 | d2 | d3) <= 1u) {
                const uint32_t b1 = 1u << ((uint32_t)r1 & 31u), b2 = 1u << ((uint32_t)r2 & 31u), b3 = 1u << ((uint32_t)r3 & 31u);
                const uint32_t lo = (1u << (q0 & 31u)) | (d1 ? 0u : b1) | (d2 ? 0u : b2) | (d3 ? 0u : b3);
                const uint32_t hi = (d1 ? b1 : 0u) | (d2 ? b2 : 0u) | (d3 ? b3 : 0u);
                const uint32_t w2[2] = {w0, w0 + 1u}, m2[2] = {lo, hi};
                sink_or_n<2>(s, w2, m2);
                return;
            }
        }
    }
    uint32_t w[4], mk[4];
#pragma unroll
    for (int c = 0; c < 4; c++) {
        const unsigned long long rel = (unsigned long long)(T)(v[c] - (T)s.id_base);
        bool ok = c < nvalid;
        if (ok && rel >= s.n_bits) { set_status(s.status, BFSC_ERR_DST_TOO_SMALL); ok = false; }
        w[c] = ok ? (uint32_t)(rel >> 5) : 0xffffffffu;
        mk[c] = ok ? 1u << ((uint32_t)rel & 31u) : 0u;
    }
#pragma unroll
    for (int c = 1; c < 4; c++)
        if (w[c] == w[c - 1]) { mk[c] |= mk[c - 1]; mk[c - 1] = 0u; }
    sink_or_n<4>(s, w, mk);
}

// Buffer of global block g: the last i with a[i] <= g (buffers without blocks are skipped), searched from a
// hint lo with a[lo] <= g (the buffer of an earlier block): gallop, then bisect. Consecutive blocks live in nearby buffers, so this touches one or two cache lines.
__device__ __forceinline__ uint32_t find_buf_from(const unsigned long long* __restrict__ a, uint32_t n_buf,
                                                  unsigned long long g, uint32_t lo) {
    uint32_t hi, step = 1;
    while (true) {
        hi = lo + step;
        if (hi >= n_buf) { hi = n_buf; break; }
        if (a[hi] > g) break;
        lo = hi; step <<= 1;
    }
    while (hi - lo > 1) {
        const uint32_t mid = (lo + hi) >> 1;
        if (a[mid] <= g) lo = mid; else hi = mid;
    }
    return lo;
}

// Plan kernels: buffer of the first block of every group of kTileBlocks blocks -> second word of the
// group's workspace entry (the hint of find_buf_from). Buffer i with blocks [first, first + nb) owns the
// groups whose first block it contains: no search. Buffers that own many groups are queued (shared
// list, kHintQueue entries) and written by the whole CTA in plan_hints_flush.
constexpr int kHintQueue = 1024;
struct HintQueue { unsigned int n; unsigned int buf[kHintQueue]; unsigned long long first[kHintQueue], nb[kHintQueue]; };

__device__ __forceinline__ void plan_hints_of(uint32_t i, unsigned long long first, unsigned long long nb,
                                              unsigned long long* __restrict__ tile_state, size_t tile_cap, HintQueue* q) {
    if (nb == 0) return;
    const unsigned long long t0 = (first + kTileBlocks - 1) / kTileBlocks, t1 = (first + nb - 1) / kTileBlocks;   // groups t0..t1
    if (t1 < t0) return;
    if (t1 - t0 < 8) {
        for (unsigned long long t = t0; t <= t1 && t < tile_cap; t++) tile_state[t * kStateStride + 1] = i;
    } else {
        const unsigned int slot = atomicAdd(&q->n, 1u);
        if (slot < (unsigned)kHintQueue) { q->buf[slot] = i; q->first[slot] = first; q->nb[slot] = nb; }
        else for (unsigned long long t = t0; t <= t1 && t < tile_cap; t++) tile_state[t * kStateStride + 1] = i;
    }
}
__device__ __forceinline__ void plan_hints_flush(unsigned long long* __restrict__ tile_state, size_t tile_cap, HintQueue* q) {
    __syncthreads();
    const unsigned int n = q->n < (unsigned)kHintQueue ? q->n : (unsigned)kHintQueue;
    const unsigned int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, nw = blockDim.x >> 5;
    for (unsigned int e = warp; e < n; e += nw) {        // one warp per queued buffer (not every warp through every entry)
        const unsigned long long t0 = (q->first[e] + kTileBlocks - 1) / kTileBlocks, t1 = (q->first[e] + q->nb[e] - 1) / kTileBlocks;
        const unsigned int b = q->buf[e];
        for (unsigned long long t = t0 + lane; t <= t1 && t < tile_cap; t += 32) tile_state[t * kStateStride + 1] = b;
    }
    __syncthreads();
    if (threadIdx.x == 0) q->n = 0;
    __syncthreads();
}
__device__ __forceinline__ uint32_t group_hint(const unsigned long long* __restrict__ tile_state, unsigned long long g) {
    return (uint32_t)tile_state[(g / kTileBlocks) * kStateStride + 1];
}

// 1024-thread exclusive scan of two u64 values with running carry (plan kernels).
struct Scan2 {
    unsigned long long a, b;
};
__device__ inline Scan2 block_scan_excl2(Scan2 v, Scan2* total, Scan2* sm /* 33 entries */) {
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = blockDim.x >> 5;
    Scan2 inc = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        unsigned long long ta = __shfl_up_sync(kFull, inc.a, o), tb = __shfl_up_sync(kFull, inc.b, o);
        if (lane >= o) { inc.a += ta; inc.b += tb; }
    }
    if (lane == 31) sm[wid] = inc;
    __syncthreads();
    if (wid == 0) {
        Scan2 w = lane < nw ? sm[lane] : Scan2{0, 0};
        Scan2 wi = w;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            unsigned long long ta = __shfl_up_sync(kFull, wi.a, o), tb = __shfl_up_sync(kFull, wi.b, o);
            if (lane >= o) { wi.a += ta; wi.b += tb; }
        }
        if (lane < nw) sm[lane] = Scan2{wi.a - w.a, wi.b - w.b};
        if (lane == 31) sm[32] = wi;
    }
    __syncthreads();
    Scan2 r{inc.a - v.a + sm[wid].a, inc.b - v.b + sm[wid].b};
    *total = sm[32];
    __syncthreads();
    return r;
}

extern unsigned long long g_launches;   // host-side launch counter (api.cu)

// Per-device launch set-up (api.cu): the SM count of the CURRENT device and a once-per-device flag table, so
// that every device of the process gets its cudaFuncSetAttribute / occupancy query (thread-safe).
constexpr int kMaxDevices = 64;
struct DeviceInfo { int device; int sms; };
bool current_device(DeviceInfo* d);      // false: no current device

// Programmatic dependent launch: a kernel launched with launch_dep may start while its predecessor in
// the stream still runs (once that one executed pdl_launch_dependents); it must execute pdl_wait
// before it touches anything the predecessor writes.
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

template <typename A>
static inline cudaError_t launch_dep(void (*kern)(A), int grid, int block, size_t smem, cudaStream_t s, const A& args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)grid); cfg.blockDim = dim3((unsigned)block);
    cfg.dynamicSmemBytes = smem; cfg.stream = s;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kern, args);
}
// The same for kernels with a plain parameter list.
template <typename... P, typename... A>
static inline cudaError_t launch_dep_v(void (*kern)(P...), int grid, int block, size_t smem, cudaStream_t s, A... args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)grid); cfg.blockDim = dim3((unsigned)block);
    cfg.dynamicSmemBytes = smem; cfg.stream = s;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kern, static_cast<P>(args)...);
}

}  // namespace bfsc

// One launch through launch_dep: its own return value decides (an earlier, unrelated error of the process is
// neither reported here nor cleared); counts the launch (calls may come from several host threads).
#define BFSC_LAUNCH(expr)                                                        \
    do {                                                                         \
        if ((expr) != cudaSuccess) return BFSC_ERR_CUDA;                         \
        __atomic_fetch_add(&::bfsc::g_launches, 1ull, __ATOMIC_RELAXED);         \
    } while (0)
