// quad_decode.cuh — decode steps D1-D4 with FOUR LANES PER BLOCK: a warp decodes 8 consecutive
// 128-ID blocks at once. lane = 4*q + l: q = block of the batch, l = lane of the quad.
// Lane l owns rows r = 4i + l, i = 0..7 (IDs 16i + 4l .. 16i + 4l + 3): per step i the quad writes
// 64 (u32) / 128 (u64) contiguous bytes, so loads and stores are coalesced 128-bit accesses, and the
// per-block scalar work (header, directory, validation) costs 1/8 of a warp instruction per block.
//
// Fast path only: blocks of at most DecStage<W>::kSpanMax 16-byte chunks (u32: b <= 20 without exceptions; u64: b <= 32),
// staged in shared memory by cp.async. Larger blocks take the warp-per-block path of block_decode.cuh.
#pragma once
#include "common.cuh"

namespace bfsc {

constexpr int kDecBlocks = 8;                 // blocks per warp batch
// Staging geometry. u32 (and the TMA variant): blocks of up to 21 chunks (336 B: b = 20) are staged, 16 warps x 2 CTAs fill
// the SM's shared memory. u64 (8 warps x 2 CTAs: room to spare): up to 33 chunks (528 B: b = 32 without exceptions; NOT
// more: a staged block is unpacked with 32-bit funnel shifts, and b = 33 starts at 34 chunks) — gaps over 2^20 between
// sorted 64-bit IDs stay on the fast path (2^24 IDs: 77 -> 40 us).
template <int W, bool kTma = false> struct DecStage {
    static constexpr int kSpanMax = (W == 64 && !kTma) ? 33 : 21;   // largest staged block, in 16-byte chunks
    static constexpr int kSlotChunks = kSpanMax + 1;               // slot stride: one chunk of slack for the unpack's second read
    static constexpr int kStageChunks = kDecBlocks * kSlotChunks;
};

__device__ __forceinline__ void dec_cp_async16(void* smem_dst, const void* gmem_src) {
    const uint32_t d = (uint32_t)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(d), "l"(gmem_src) : "memory");
}
__device__ __forceinline__ void dec_cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }

// D1, bulk variant: mbarrier + cp.async.bulk (TMA), one copy per warp batch, issued by one lane.
__device__ __forceinline__ void dec_mbar_init(unsigned long long* b, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"((uint32_t)__cvta_generic_to_shared(b)), "r"(count) : "memory");
}
__device__ __forceinline__ void dec_fence_mbar_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void dec_mbar_expect_tx(unsigned long long* b, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"((uint32_t)__cvta_generic_to_shared(b)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void dec_bulk_load(void* sdst, const void* gsrc, uint32_t bytes, unsigned long long* b) {   // 16-byte aligned, multiple of 16
    asm volatile("cp.async.bulk.shared::cta.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"((uint32_t)__cvta_generic_to_shared(sdst)),
                 "l"(gsrc), "r"(bytes), "r"((uint32_t)__cvta_generic_to_shared(b)) : "memory");
}
__device__ __forceinline__ void dec_mbar_wait(unsigned long long* b, uint32_t parity) {      // whole warp
    const uint32_t addr = (uint32_t)__cvta_generic_to_shared(b);
    uint32_t ok;
    do {
        asm volatile("{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n selp.u32 %0, 1, 0, p;\n}"
                     : "=r"(ok) : "r"(addr), "r"(parity) : "memory");
    } while (!ok);
}

// D1: stage the quad's block (span16 <= kSpanMax chunks at blk) into its slot; lane l copies chunks l, l+4, ...
template <int kSpanMax>
__device__ __forceinline__ void quad_stage_block(uint4* __restrict__ slot, const unsigned char* __restrict__ blk,
                                                 uint32_t span16, int l) {
    const uint4* src = reinterpret_cast<const uint4*>(blk);
#pragma unroll
    for (int i = 0; i < (kSpanMax + 3) / 4; i++) {
        const uint32_t c = 4 * i + l;
        if (c < span16) dec_cp_async16(slot + c, src + c);
    }
}

// D3 (first half): exceptions go through a per-warp patch table (128 entries per block, all zero between
// uses): the quad scatters high << b at each position here; quad_decode_rows ORs the entries in;
// quad_patch_clear zeroes them again. e = staged exception area. Returns false on a malformed position
// (>= 128, or not above its predecessor: FORMAT.md §4).
template <int W>
__device__ __forceinline__ bool quad_patch_scatter(typename IdT<W>::T* __restrict__ tab /* the quad's 128 entries */,
                                                   const unsigned char* __restrict__ e, uint32_t b, uint32_t n_exc, int l) {
    using T = typename IdT<W>::T;
    constexpr uint32_t E = W / 8;
    const T* high = reinterpret_cast<const T*>(e + ((n_exc + E - 1) & ~(E - 1)));
    bool ok = true;
    for (uint32_t x = l; x < n_exc; x += 4) {
        const uint32_t pos = e[x];
        if (pos >= (uint32_t)kBlk || (x > 0 && pos <= e[x - 1])) ok = false;   // FORMAT.md §4: < 128, strictly ascending
        else tab[pos] = high[x] << b;
    }
    return ok;
}
template <int W>
__device__ __forceinline__ void quad_patch_clear(typename IdT<W>::T* __restrict__ tab, const unsigned char* __restrict__ e,
                                                 uint32_t n_exc, int l) {
    for (uint32_t x = l; x < n_exc; x += 4) {
        const uint32_t pos = e[x];
        if (pos < (uint32_t)kBlk) tab[pos] = 0;
    }
}

// D2 + D3 + D4, one row step at a time (nothing but the running sum is carried between steps):
//   D2  low parts of row r = 4i + l from the staged payload P (b <= 16 vectors of 128 bits; FORMAT.md §2
//       "Payload"): row r's values sit at bits [r b, r b + b) of each column stream; the second vector
//       read may be one past the payload (slack chunk / exception area): its bits are masked off;
//   D3  OR of the patch table's row (only if some block of the warp has exceptions);
//   D4  inclusive scan: prefix inside the row, inclusive scan of the row sums over the quad, running
//       carry over the steps (order of the IDs: i major, then lane, then column); + base, mod 2^W;
//       128-bit stores of the first m IDs.
// kBits: the IDs are not stored; their bits go into the bitmap of `sink` (FORMAT.md §9).
template <int W, bool kWin, bool kBits = false>
__device__ __forceinline__ void quad_decode_rows(const uint4* __restrict__ P, uint32_t b,
                                                 const typename IdT<W>::T* __restrict__ tab, bool patch,
                                                 typename IdT<W>::T base, typename IdT<W>::T* __restrict__ x, int m, int l,
                                                 const BitSink& sink = BitSink{nullptr, 0, 0, nullptr, nullptr}) {
    using T = typename IdT<W>::T;
    const uint32_t mask = b >= 32u ? 0xffffffffu : (1u << b) - 1u;       // (b <= 32 here: larger blocks are not staged)
    uint32_t bit = (uint32_t)l * b;
    T carry = base;
    const bool vec_ok = (m == kBlk) && ((reinterpret_cast<uintptr_t>(x) & 15) == 0);
    const bool vec = __all_sync(kFull, vec_ok || m <= 0);
    // General path (some block of the warp is ragged or its output is not 16-byte aligned — buffers of a
    // batch start at any element). kWin (batch calls): the row is shifted by e elements through the quad so
    // that every lane still writes one ALIGNED 16/32-byte window (prev row's last e values | this row's
    // first 4 - e); full-sector stores matter: 4- and 8-byte stores quadruple the L2 write requests.
    // !kWin (single stream: only the warp with the ragged last block gets here): guarded element stores.
    const int lane = threadIdx.x & 31;
    const int e = (int)((reinterpret_cast<uintptr_t>(x) & 15) / sizeof(T));
    const int src = (l == 0) ? lane + 3 : lane - 1;                     // owner of the previous row
    T q1 = 0, q2 = 0, q3 = 0;                                            // this lane's previous row step
#pragma unroll
    for (int i = 0; i < 8; i++) {
        const uint32_t k0 = bit >> 5, sh = bit & 31u;
        const uint4 lo = P[k0], hi = P[k0 + 1];                          // (loading hi only when a value straddles the chunk: +9 % instructions, same time)
        bit += 4u * b;
        T v0 = __funnelshift_r(lo.x, hi.x, sh) & mask, v1 = __funnelshift_r(lo.y, hi.y, sh) & mask;
        T v2 = __funnelshift_r(lo.z, hi.z, sh) & mask, v3 = __funnelshift_r(lo.w, hi.w, sh) & mask;
        if (patch) {
            if constexpr (W == 32) {
                const uint4 t = reinterpret_cast<const uint4*>(tab)[4 * i + l];
                v0 |= t.x; v1 |= t.y; v2 |= t.z; v3 |= t.w;
            } else {
                const ulonglong2 t0 = reinterpret_cast<const ulonglong2*>(tab)[2 * (4 * i + l)];
                const ulonglong2 t1 = reinterpret_cast<const ulonglong2*>(tab)[2 * (4 * i + l) + 1];
                v0 |= t0.x; v1 |= t0.y; v2 |= t1.x; v3 |= t1.y;
            }
        }
        v1 += v0; v2 += v1; v3 += v2;                                    // prefix inside the row
        T inc = v3;                                                      // inclusive scan of the row sums over the quad
        T t = __shfl_up_sync(kFull, inc, 1, 4);
        if (l >= 1) inc += t;
        t = __shfl_up_sync(kFull, inc, 2, 4);
        if (l >= 2) inc += t;
        const T tot = __shfl_sync(kFull, inc, 3, 4);
        const T off = carry + (inc - v3);
        carry += tot;
        v0 += off; v1 += off; v2 += off; v3 += off;
        if constexpr (kBits) {
            set_bits4<T>(sink, v0, v1, v2, v3, m - (16 * i + 4 * l));
        } else if (vec) {
            if (m > 0) {
                if constexpr (W == 32) {
                    __stcs(reinterpret_cast<uint4*>(x) + 4 * i + l, make_uint4(v0, v1, v2, v3));
                } else {
                    ulonglong2* p = reinterpret_cast<ulonglong2*>(x) + 2 * (4 * i + l);
                    __stcs(p, make_ulonglong2(v0, v1));
                    __stcs(p + 1, make_ulonglong2(v2, v3));
                }
            }
        } else if constexpr (!kWin) {
            const int jx = 16 * i + 4 * l;
            if (jx < m) x[jx] = v0;
            if (jx + 1 < m) x[jx + 1] = v1;
            if (jx + 2 < m) x[jx + 2] = v2;
            if (jx + 3 < m) x[jx + 3] = v3;
        } else {
            // previous row's v1..v3: lane l-1 of this step, or lane 3 of the previous step (which publishes q*)
            const T p1 = __shfl_sync(kFull, l == 3 ? q1 : v1, src), p2 = __shfl_sync(kFull, l == 3 ? q2 : v2, src);
            const T p3 = __shfl_sync(kFull, l == 3 ? q3 : v3, src);
            q1 = v1; q2 = v2; q3 = v3;
            const T c0 = e == 0 ? v0 : (e == 1 ? p3 : (e == 2 ? p2 : p1));
            const T c1 = e == 0 ? v1 : (e == 1 ? v0 : (e == 2 ? p3 : p2));
            const T c2 = e == 0 ? v2 : (e == 1 ? v1 : (e == 2 ? v0 : p3));
            const T c3 = e == 0 ? v3 : (e == 1 ? v2 : (e == 2 ? v1 : v0));
            const int j0 = 16 * i + 4 * l - e;                           // first element of the window
            T* w = x + j0;                                               // 16-byte aligned
            if (j0 >= 0 && j0 + 3 < m) {
                if constexpr (W == 32) {
                    __stcs(reinterpret_cast<uint4*>(w), make_uint4(c0, c1, c2, c3));
                } else {
                    __stcs(reinterpret_cast<ulonglong2*>(w), make_ulonglong2(c0, c1));
                    __stcs(reinterpret_cast<ulonglong2*>(w) + 1, make_ulonglong2(c2, c3));
                }
            } else {
                if (j0 >= 0 && j0 < m) w[0] = c0;
                if (j0 + 1 >= 0 && j0 + 1 < m) w[1] = c1;
                if (j0 + 2 >= 0 && j0 + 2 < m) w[2] = c2;
                if (j0 + 3 < m) w[3] = c3;                               // j0 + 3 >= 0 always
            }
            if (i == 7 && l == 3) {                                      // the block's last e elements
                if (e >= 1 && 127 < m) x[127] = v3;
                if (e >= 2 && 126 < m) x[126] = v2;
                if (e >= 3 && 125 < m) x[125] = v1;
            }
        }
    }
}

}  // namespace bfsc
