// bitmap_stage.cuh — E1 for a frontier given as a bitmap (FORMAT.md §9): the IDs of a
// block are the positions of 128 consecutive set bits. k_bm_starts has recorded where every block begins (bit index of
// its first ID); a worker warp stages the bitmap words of its 8 blocks by cp.async one tile ahead (landing area) and
// expands them into the quads' raw-ID slots, where E1-E4 find them as if they had been loaded from an ID array.
#pragma once
#include "quad_encode.cuh"

namespace bfsc {

// Whole warp. st: the tile's block starts (entry j: first bit of block j of the tile, entry 64: end of its last block);
// the warp's blocks are 8 * warp .. 8 * warp + 7. The words between the first bit of the first and the last bit of the
// last block go to the landing area as 16-byte chunks, one per lane, if kLand chunks hold them (else bm_expand reads
// the bitmap itself). The bitmap is readable up to a multiple of 16 bytes (include/bfsc.h).
template <int kLand>
__device__ __forceinline__ void bm_prefetch(uint4* __restrict__ land, const uint32_t* __restrict__ bitmap,
                                            const uint32_t* __restrict__ st, int warp, int lane) {
    const uint32_t s0 = st[kQuadBlocks * warp], e0 = st[kQuadBlocks * warp + kQuadBlocks];
    if (e0 <= s0) return;
    const uint32_t c_lo = s0 >> 7, n = ((e0 - 1u) >> 7) - c_lo + 1u;
    if (n <= (uint32_t)kLand && (uint32_t)lane < n) cp_async16(land + lane, reinterpret_cast<const uint4*>(bitmap) + c_lo + lane);
}

// The quad's block: its set bits -> raw[0 .. m) = id_base + bit index, ascending. Lanes of a quad take the block's words
// four at a time (lane l: word w + l); ranks by a scan of the popcounts over the quad. Every lane of the warp calls
// (quads loop on their own: the shuffles stay inside the quad).
template <typename T, int kLand>
__device__ __forceinline__ void bm_expand(T* __restrict__ raw, const uint32_t* __restrict__ st, int warp, int q, int l,
                                          const uint4* __restrict__ land, const uint32_t* __restrict__ bitmap,
                                          unsigned long long id_base) {
    const uint32_t s = st[kQuadBlocks * warp + q], e = st[kQuadBlocks * warp + q + 1];
    if (e <= s) return;
    const uint32_t s0 = st[kQuadBlocks * warp], e0 = st[kQuadBlocks * warp + kQuadBlocks];
    const uint32_t c_lo = s0 >> 7;
    const bool landed = ((e0 - 1u) >> 7) - c_lo + 1u <= (uint32_t)kLand;
    const uint32_t* words = landed ? reinterpret_cast<const uint32_t*>(land) - 4ull * c_lo : bitmap;   // indexed by word number
    const uint32_t w_first = s >> 5, w_last = (e - 1u) >> 5;
    const uint32_t qmask = 0xfu << (4 * q);
    uint32_t rank = 0;
    if (!landed) {
        // A sparse batch (more than kLand chunks: under one ID in 32 bits on average): its words come from global memory,
        // SIXTEEN per quad and trip (one 128-bit load per lane), and a trip without a set bit costs a vote, not a scan —
        // one word per lane and trip made a block of a 0.2 % dense bitmap (2000 words) five hundred dependent trips long.
        for (uint32_t w = w_first & ~3u; w <= w_last && w >= (w_first & ~3u); w += 16) {
            const uint32_t w4 = w + 4u * (uint32_t)l;
            uint4 v = make_uint4(0u, 0u, 0u, 0u);
            if (w4 <= w_last && w4 >= w) v = *reinterpret_cast<const uint4*>(bitmap + w4);
            uint32_t xs[4] = {v.x, v.y, v.z, v.w};
            uint32_t c = 0;
#pragma unroll
            for (int t = 0; t < 4; t++) {
                const uint32_t wi = w4 + (uint32_t)t;
                if (wi < w_first || wi > w_last || wi < w) xs[t] = 0u;
                if (wi == w_first) xs[t] &= 0xffffffffu << (s & 31u);
                if (wi == w_last && (e & 31u)) xs[t] &= (1u << (e & 31u)) - 1u;
                c += (uint32_t)__popc(xs[t]);
            }
            if (!__any_sync(qmask, c != 0u)) continue;
            uint32_t inc = c, y;
            y = __shfl_up_sync(qmask, inc, 1, 4); if (l >= 1) inc += y;
            y = __shfl_up_sync(qmask, inc, 2, 4); if (l >= 2) inc += y;
            T* out = raw + (rank + inc);                             // behind this lane's last ID: filled from the top down
            rank += __shfl_sync(qmask, inc, 3, 4);
#pragma unroll
            for (int t = 3; t >= 0; t--) {
                uint32_t x = xs[t];
                const T id0 = (T)(id_base + 32ull * (w4 + (uint32_t)t));
                while (x) {
                    uint32_t b;
                    asm("bfind.u32 %0, %1;" : "=r"(b) : "r"(x));
                    BFSC_CHECK(out - 1 >= raw && out - 1 < raw + kBlk);
                    *--out = id0 + (T)b;
                    x &= ~(1u << (b & 31u));
                }
            }
        }
        return;
    }
    for (uint32_t w = w_first; w <= w_last && w >= w_first; w += 4) {
        const uint32_t wi = w + (uint32_t)l;
        uint32_t x = (wi <= w_last && wi >= w) ? words[wi] : 0u;
        if (wi == w_first) x &= 0xffffffffu << (s & 31u);
        if (wi == w_last && (e & 31u)) x &= (1u << (e & 31u)) - 1u;
        const uint32_t c = (uint32_t)__popc(x);
        uint32_t inc = c, y;
        y = __shfl_up_sync(qmask, inc, 1, 4); if (l >= 1) inc += y;
        y = __shfl_up_sync(qmask, inc, 2, 4); if (l >= 2) inc += y;
        // the word's set bits from the top down (one bfind per bit, no bit reversal), written backwards from the rank
        // behind the word's last ID; four bits per trip, the stores predicated
        T* out = raw + (rank + inc);
        rank += __shfl_sync(qmask, inc, 3, 4);
        const T id0 = (T)(id_base + 32ull * wi);
        while (x) {
#pragma unroll
            for (int u = 1; u <= 4; u++) {
                uint32_t b;
                asm("bfind.u32 %0, %1;" : "=r"(b) : "r"(x));               // 0xffffffff for x == 0
                BFSC_CHECK(!x || (out - u >= raw && out - u < raw + kBlk));
                if (x) out[-u] = id0 + (T)b;
                x &= ~(1u << (b & 31u));
            }
            out -= 4;
        }
    }
}

}  // namespace bfsc
