// block_decode.cuh — per-block decode steps D2 (unpack), D3 (patch), D4 (scan + store) of
// SURVEY.md §8(a). warp = block, lane r produces row r = IDs 4r..4r+3.
#pragma once
#include "common.cuh"

namespace bfsc {

// Unpack the lane's 4 low parts from a payload of b 128-bit vectors (FORMAT.md §2 "Payload").
// P may point to global or shared memory; reads stay inside [P, P + 16*b).
template <int W>
__device__ __forceinline__ void unpack_rows(const uint4* __restrict__ P, uint32_t b,
                                            typename IdT<W>::T d[4]) {
    using T = typename IdT<W>::T;
    const uint32_t lane = lane_id();
    if (b == 0) { d[0] = d[1] = d[2] = d[3] = 0; return; }
    const uint32_t bit = lane * b, k0 = bit >> 5, sh = bit & 31;
    if (b <= 32) {
        const uint4 lo = P[k0];
        uint4 hi = make_uint4(0, 0, 0, 0);
        if (sh + b > 32) hi = P[k0 + 1];            // then k0+1 < b
        const uint32_t mask = (b == 32) ? 0xffffffffu : ((1u << b) - 1u);
        d[0] = (T)(__funnelshift_r(lo.x, hi.x, sh) & mask);
        d[1] = (T)(__funnelshift_r(lo.y, hi.y, sh) & mask);
        d[2] = (T)(__funnelshift_r(lo.z, hi.z, sh) & mask);
        d[3] = (T)(__funnelshift_r(lo.w, hi.w, sh) & mask);
    } else if constexpr (W == 64) {                 // a value spans 2 or 3 words
        const uint4 w0 = P[k0];
        const uint4 w1 = P[k0 + 1];                 // sh + b > 32 always here
        uint4 w2 = make_uint4(0, 0, 0, 0);
        if (sh + b > 64) w2 = P[k0 + 2];
        const uint64_t mask = (b == 64) ? ~0ull : ((1ull << b) - 1ull);
        const uint32_t a0[4] = {w0.x, w0.y, w0.z, w0.w}, a1[4] = {w1.x, w1.y, w1.z, w1.w},
                       a2[4] = {w2.x, w2.y, w2.z, w2.w};
#pragma unroll
        for (int c = 0; c < 4; c++) {
            uint64_t v = ((uint64_t)a1[c] << 32 | a0[c]) >> sh;
            if (sh) v |= (uint64_t)a2[c] << (64 - sh);
            d[c] = v & mask;
        }
    }
}

// D3: OR the exceptions' high parts into place. e = exception area (pos bytes, pad, highs).
// Returns false on a malformed position (>= 128, or not above its predecessor).
template <int W>
__device__ __forceinline__ bool patch_rows(const unsigned char* __restrict__ e, uint32_t b, uint32_t n_exc,
                                           typename IdT<W>::T d[4]) {
    using T = typename IdT<W>::T;
    constexpr uint32_t E = W / 8;
    const uint32_t lane = lane_id();
    const T* high = reinterpret_cast<const T*>(e + ((n_exc + E - 1) & ~(E - 1)));
    bool ok = true;
    for (uint32_t i0 = 0; i0 < n_exc; i0 += 32) {
        const uint32_t i = i0 + lane;
        uint32_t pos = 0xffffffffu; T hv = 0;
        if (i < n_exc) {
            pos = e[i]; hv = high[i];
            if (pos >= (uint32_t)kBlk || (i > 0 && pos <= e[i - 1])) ok = false;   // FORMAT.md §4: < 128, strictly ascending
        }
        const uint32_t cnt = min(32u, n_exc - i0);
        for (uint32_t q = 0; q < cnt; q++) {
            const uint32_t p = __shfl_sync(kFull, pos, q);
            const T h = __shfl_sync(kFull, hv, q);
            if ((p >> 2) == lane && b < (uint32_t)W) {
                const T add = h << b;
                const uint32_t c = p & 3;
                d[0] |= (c == 0) ? add : (T)0; d[1] |= (c == 1) ? add : (T)0;
                d[2] |= (c == 2) ? add : (T)0; d[3] |= (c == 3) ? add : (T)0;
            }
        }
    }
    return __all_sync(kFull, ok);
}

// D4: inclusive scan of the 128 deltas (4 local adds + warp scan of row totals) + base, then store
// the first m IDs. x: block's first output ID.
template <int W, bool kBits = false>
__device__ __forceinline__ void scan_store(typename IdT<W>::T d[4], typename IdT<W>::T base,
                                           typename IdT<W>::T* __restrict__ x, int m,
                                           const BitSink& sink = BitSink{nullptr, 0, 0, nullptr, nullptr}) {
    using T = typename IdT<W>::T;
    const int lane = lane_id();
    d[1] += d[0]; d[2] += d[1]; d[3] += d[2];
    T inc = d[3];
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        T t = __shfl_up_sync(kFull, inc, o);
        if (lane >= o) inc += t;
    }
    const T off = base + (inc - d[3]);
    d[0] += off; d[1] += off; d[2] += off; d[3] += off;
    if constexpr (kBits) {
        set_bits4<T>(sink, d[0], d[1], d[2], d[3], m - 4 * lane);
        return;
    }
    const bool vec_ok = (m == kBlk) && ((reinterpret_cast<uintptr_t>(x) & 15) == 0);
    if (vec_ok) {
        if constexpr (W == 32) {
            __stcs(reinterpret_cast<uint4*>(x) + lane, make_uint4(d[0], d[1], d[2], d[3]));
        } else {
            ulonglong2* p = reinterpret_cast<ulonglong2*>(x) + 2 * lane;
            __stcs(p, make_ulonglong2(d[0], d[1]));
            __stcs(p + 1, make_ulonglong2(d[2], d[3]));
        }
    } else {
#pragma unroll
        for (int c = 0; c < 4; c++) if (4 * lane + c < m) x[4 * lane + c] = d[c];
    }
}

}  // namespace bfsc
