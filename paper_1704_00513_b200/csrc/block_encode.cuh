// block_encode.cuh — per-block (128 IDs = one warp) encode steps E1, E2, E4 of SURVEY.md §8(a).
// Mapping: warp = block, lane r holds row r = IDs 4r..4r+3 (one 128-bit load for u32).
#pragma once
#include "common.cuh"

namespace bfsc {

template <int W> struct IdT;
template <> struct IdT<32> { using T = uint32_t; };
template <> struct IdT<64> { using T = uint64_t; };

// ceil(2^32 / b) for b = 2..64 ([0], [1] unused): floor(num / b) == umulhi(num, kRecip[b]) for num < 2^12
static __constant__ uint32_t kRecip[65] = {
    0u, 0u, 2147483648u, 1431655766u, 1073741824u, 858993460u, 715827883u, 613566757u, 536870912u,
    477218589u, 429496730u, 390451573u, 357913942u, 330382100u, 306783379u, 286331154u, 268435456u,
    252645136u, 238609295u, 226050911u, 214748365u, 204522253u, 195225787u, 186737709u, 178956971u,
    171798692u, 165191050u, 159072863u, 153391690u, 148102321u, 143165577u, 138547333u, 134217728u,
    130150525u, 126322568u, 122713352u, 119304648u, 116080198u, 113025456u, 110127367u, 107374183u,
    104755300u, 102261127u, 99882961u, 97612894u, 95443718u, 93368855u, 91382283u, 89478486u,
    87652394u, 85899346u, 84215046u, 82595525u, 81037119u, 79536432u, 78090315u, 76695845u,
    75350304u, 74051161u, 72796056u, 71582789u, 70409300u, 69273667u, 68174085u, 67108864u};

__device__ __forceinline__ uint32_t div_small(uint32_t num, uint32_t b) {
    return b == 1 ? num : __umulhi(num, kRecip[b]);
}

// ---- E1: load + delta (store the distances between successive elements) ----
// x: first ID of the block; m valid IDs (1..128). v[c] = ID 4*lane+c (0 beyond m).
template <int W>
__device__ __forceinline__ void load_rows(const typename IdT<W>::T* __restrict__ x, int m,
                                          typename IdT<W>::T v[4]) {
    using T = typename IdT<W>::T;
    const int lane = lane_id();
    const bool vec_ok = (m == kBlk) && ((reinterpret_cast<uintptr_t>(x) & 15) == 0);
    if (vec_ok) {
        if constexpr (W == 32) {
            uint4 q = __ldcs(reinterpret_cast<const uint4*>(x) + lane);
            v[0] = q.x; v[1] = q.y; v[2] = q.z; v[3] = q.w;
        } else {
            const ulonglong2* p = reinterpret_cast<const ulonglong2*>(x) + 2 * lane;
            ulonglong2 a = __ldcs(p), b = __ldcs(p + 1);
            v[0] = a.x; v[1] = a.y; v[2] = b.x; v[3] = b.y;
        }
    } else {
#pragma unroll
        for (int c = 0; c < 4; c++) v[c] = (4 * lane + c < m) ? x[4 * lane + c] : (T)0;
    }
}

// Same as load_rows, but with the default (evict-normal) cache policy: used by the first pass over a
// tile, whose second pass re-reads the data from L2.
template <int W>
__device__ __forceinline__ void load_rows_keep(const typename IdT<W>::T* __restrict__ x, int m,
                                               typename IdT<W>::T v[4]) {
    using T = typename IdT<W>::T;
    const int lane = lane_id();
    const bool vec_ok = (m == kBlk) && ((reinterpret_cast<uintptr_t>(x) & 15) == 0);
    if (vec_ok) {
        if constexpr (W == 32) {
            uint4 q = __ldg(reinterpret_cast<const uint4*>(x) + lane);
            v[0] = q.x; v[1] = q.y; v[2] = q.z; v[3] = q.w;
        } else {
            const ulonglong2* p = reinterpret_cast<const ulonglong2*>(x) + 2 * lane;
            ulonglong2 a = __ldg(p), b = __ldg(p + 1);
            v[0] = a.x; v[1] = a.y; v[2] = b.x; v[3] = b.y;
        }
    } else {
#pragma unroll
        for (int c = 0; c < 4; c++) v[c] = (4 * lane + c < m) ? x[4 * lane + c] : (T)0;
    }
}

// d[c] = delta of ID 4*lane+c (d_0 = 0, zero beyond m). Returns base = first ID (all lanes).
template <int W>
__device__ __forceinline__ typename IdT<W>::T deltas(const typename IdT<W>::T v[4], int m,
                                                     typename IdT<W>::T d[4]) {
    using T = typename IdT<W>::T;
    const int lane = lane_id();
    T prev = __shfl_up_sync(kFull, v[3], 1);
    if (lane == 0) prev = v[0];
    d[0] = v[0] - prev; d[1] = v[1] - v[0]; d[2] = v[2] - v[1]; d[3] = v[3] - v[2];
    if (m < kBlk) {
#pragma unroll
        for (int c = 0; c < 4; c++) if (4 * lane + c >= m) d[c] = 0;
    }
    return __shfl_sync(kFull, v[0], 0);
}

// ---- E2: width + choice of b ---------------------------------------------------------
// Input: widths of the lane's 4 deltas (eq. 6: bit length). Output key =
// block_bytes << 14 | (64 - b) << 7 | n_exc of the canonical b (FORMAT.md §2: argmin of the exact
// block size over b in 0..maxw, ties to the largest b). Exact for every input:
// windows of 9 candidate widths [top-8, top] are evaluated with byte-packed counters summed by
// __reduce_add_sync; a window chain stops when the exception area implied by the values above
// the window already costs at least the best size found (sizes are monotone in n_exc), and
// skips widths that no value has (such a b is dominated by b-1: same exceptions, less payload).
template <int W>
__device__ __forceinline__ uint32_t choose_b(const int w[4]) {
    const int lane = lane_id();
    int top = __reduce_max_sync(kFull, (unsigned)max(max(w[0], w[1]), max(w[2], w[3])));
    uint32_t cnt_above = 0, best = 0xffffffffu;
    while (true) {
        uint32_t S = 0;
#pragma unroll
        for (int c = 0; c < 4; c++) {
            int t = top - w[c];                     // value is an exception for b = top - s iff t < s
            if (t >= 0) S += shl32(0x11111111u, 4u * (uint32_t)t);   // nibble i (s = i+1) set iff i >= t
        }
        uint32_t lo = S & 0x0f0f0f0fu, hi = (S >> 4) & 0x0f0f0f0fu; // per-lane counts <= 4, warp sums <= 128
        lo = __reduce_add_sync(kFull, lo);
        hi = __reduce_add_sync(kFull, hi);
        uint32_t key = 0xffffffffu;
        if (lane <= 8 && lane <= top) {             // lane s evaluates b = top - s
            uint32_t n = cnt_above;
            if (lane > 0) {
                int i = lane - 1;
                n += (((i & 1) ? hi : lo) >> (8 * (i >> 1))) & 0xffu;
            }
            uint32_t b = (uint32_t)(top - lane);
            uint32_t cost = 16u + 16u * b + exc_bytes<W>(n);
            key = (cost << 14) | ((64u - b) << 7) | n;
        }
        key = __reduce_min_sync(kFull, key);
        best = min(best, key);
        if (top <= 8) break;                        // candidates down to b = 0 were covered
        uint32_t n_bot = cnt_above + ((hi >> 24) & 0xffu);          // exceptions at b = top - 8
        if (16u + exc_bytes<W>(n_bot) >= (best >> 14)) break;       // nothing below can be smaller
        int below = 0;
#pragma unroll
        for (int c = 0; c < 4; c++) if (w[c] <= top - 8) below = max(below, w[c]);
        top = __reduce_max_sync(kFull, (unsigned)below);
        cnt_above = n_bot;
    }
    return best;
}

// ---- E4: pack + emit -----------------------------------------------------------------
// Per-warp shared staging: the whole block is assembled in shared memory and leaves with
// 128-bit coalesced stores.
template <int W>
struct EncStage {
    static constexpr int kExcMax = (W == 32) ? 640 : 1152;          // exc_bytes(127)
    static constexpr int kOutBytes = 16 + 16 * W + kExcMax;
    alignas(16) typename IdT<W>::T vals[kBlk];                       // masked low parts, row-major (j = 4r+c)
    alignas(16) unsigned char out[kOutBytes];
};

// Assemble block (base, b, n_exc, deltas d[4] per lane) into st.out; returns its byte count.
template <int W>
__device__ __forceinline__ uint32_t pack_block_to(typename IdT<W>::T* __restrict__ vals, unsigned char* __restrict__ out,
                                                  const typename IdT<W>::T d[4], typename IdT<W>::T base,
                                                  uint32_t b, uint32_t n_exc) {
    using T = typename IdT<W>::T;
    const int lane = lane_id();
    uint32_t* out32 = reinterpret_cast<uint32_t*>(out);
    if (lane == 0) {
        reinterpret_cast<unsigned long long*>(out)[0] = (unsigned long long)base;
        reinterpret_cast<unsigned long long*>(out)[1] = (unsigned long long)(b | (n_exc << 8));
    }
    const uint32_t eb = exc_bytes<W>(n_exc);
    const uint32_t total = 16u + 16u * b + eb;
    if (b > 0) {
        T mask = (b >= (uint32_t)W) ? ~(T)0 : (((T)1 << b) - 1);
        if constexpr (W == 32) {
            reinterpret_cast<uint4*>(vals)[lane] = make_uint4(d[0] & mask, d[1] & mask, d[2] & mask, d[3] & mask);
        } else {
            reinterpret_cast<ulonglong2*>(vals)[2 * lane] = make_ulonglong2(d[0] & mask, d[1] & mask);
            reinterpret_cast<ulonglong2*>(vals)[2 * lane + 1] = make_ulonglong2(d[2] & mask, d[3] & mask);
        }
    }
    if (n_exc > 0) {                                // zero the exception area (pads must be 0)
        uint4* z = reinterpret_cast<uint4*>(out + 16 + 16 * b);
        for (uint32_t i = lane; i < eb / 16; i += 32) z[i] = make_uint4(0, 0, 0, 0);
    }
    __syncwarp();
    // payload: word o = 4k+c is bits [32k, 32k+32) of column c's stream (row r at bits [r*b, r*b+b))
    const uint32_t nwords = 4u * b;
    for (uint32_t o = lane; o < nwords; o += 32) {
        const uint32_t k = o >> 2, c = o & 3;
        const uint32_t r_lo = div_small(32u * k, b);
        const uint32_t r_hi = min(31u, div_small(32u * k + 31u, b));
        uint32_t word = 0;
        for (uint32_t r = r_lo; r <= r_hi; r++) {
            const T val = vals[4 * r + c];
            const int pos = (int)(r * b) - (int)(32u * k);
            if constexpr (W == 32) word |= (pos >= 0) ? (val << pos) : (val >> (-pos));
            else word |= (pos >= 0) ? (uint32_t)(val << pos) : (uint32_t)shr64(val, (uint32_t)(-pos));
        }
        out32[4 + o] = word;
    }
    if (n_exc > 0) {                                // exceptions: ascending position = (row, column) order
        unsigned char* e = out + 16 + 16 * b;
        constexpr uint32_t E = W / 8;
        T* high = reinterpret_cast<T*>(e + ((n_exc + E - 1) & ~(E - 1)));
        bool f[4];
        uint32_t before = 0;
#pragma unroll
        for (int c = 0; c < 4; c++) {
            f[c] = (b < (uint32_t)W) && ((d[c] >> b) != 0);
            uint32_t bal = __ballot_sync(kFull, f[c]);
            before += __popc(bal & ((1u << lane) - 1u));
        }
#pragma unroll
        for (int c = 0; c < 4; c++) {
            if (f[c]) {
                e[before] = (unsigned char)(4 * lane + c);
                high[before] = d[c] >> b;
                before++;
            }
        }
    }
    __syncwarp();
    return total;
}

template <int W>
__device__ __forceinline__ uint32_t pack_block(EncStage<W>& st, const typename IdT<W>::T d[4],
                                               typename IdT<W>::T base, uint32_t b, uint32_t n_exc) {
    return pack_block_to<W>(st.vals, st.out, d, base, b, n_exc);
}

// Copy an assembled block to global memory (dst 16-byte aligned) with 128-bit stores.
template <int W>
__device__ __forceinline__ void store_block(const EncStage<W>& st, unsigned char* __restrict__ dst, uint32_t total) {
    const uint4* s = reinterpret_cast<const uint4*>(st.out);
    uint4* d4 = reinterpret_cast<uint4*>(dst);
    for (uint32_t i = lane_id(); i < total / 16; i += 32) __stcs(d4 + i, s[i]);
}

template <int W>
__device__ __forceinline__ void widths_of(const typename IdT<W>::T d[4], int w[4]) {
#pragma unroll
    for (int c = 0; c < 4; c++) {
        if constexpr (W == 32) w[c] = width32(d[c]); else w[c] = width64(d[c]);
    }
}

}  // namespace bfsc
