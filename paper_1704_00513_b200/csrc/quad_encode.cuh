// quad_encode.cuh — encode steps E1, E2, E4 with FOUR LANES PER BLOCK: a warp works on 8
// consecutive 128-ID blocks at once ("batch"). lane = 4*q + l: q = block of the batch, l = lane
// of the quad. Per-block scalar work (sizes, offsets, headers) then costs 1/8 of a warp
// instruction per block instead of a whole one, and nothing needs a full-warp reduction.
//
// Two ownerships of a block's 128 values (j = 4r + c, row r = 0..31, column c = 0..3):
//   row owner   : lane l holds rows r = 4i + l, i = 0..7 (v[i][c] = x[16i + 4l + c]): the quad
//                 reads 64 contiguous bytes per load instruction (128-bit loads, coalesced);
//   column owner: lane c packs column c's bit stream (FORMAT.md payload) sequentially from the
//                 staged values in shared memory.
#pragma once
#include "block_encode.cuh"

namespace bfsc {

constexpr int kQuadBlocks = 8;                       // blocks per warp batch
constexpr int kValStride = 132;                      // words between blocks' staged rows (== 4 mod 32: conflict-free column reads)

__device__ __forceinline__ int quad_q() { return (threadIdx.x & 31) >> 2; }
__device__ __forceinline__ int quad_l() { return threadIdx.x & 3; }

template <typename DT> __device__ __forceinline__ int bitlen(DT v);
template <> __device__ __forceinline__ int bitlen<uint32_t>(uint32_t v) { return 32 - __clz(v); }
template <> __device__ __forceinline__ int bitlen<uint64_t>(uint64_t v) { return 64 - __clzll(v); }

template <typename DT> __device__ __forceinline__ DT shr_clamp(DT v, uint32_t s);
template <> __device__ __forceinline__ uint32_t shr_clamp<uint32_t>(uint32_t v, uint32_t s) { return shr32(v, s); }
template <> __device__ __forceinline__ uint64_t shr_clamp<uint64_t>(uint64_t v, uint32_t s) { return shr64(v, s); }

// ---- E1: row-owner load of the quad's block. x = block's first ID, m = valid IDs (0..128).
template <int W>
__device__ __forceinline__ void quad_load(const typename IdT<W>::T* __restrict__ x, int m, bool keep_in_l2,
                                          typename IdT<W>::T (&v)[8][4]) {
    using T = typename IdT<W>::T;
    const int l = quad_l();
    const bool fast = (m == kBlk) && ((reinterpret_cast<uintptr_t>(x) & 15) == 0);
    if (__all_sync(kFull, fast)) {
        if constexpr (W == 32) {
            const uint4* p = reinterpret_cast<const uint4*>(x) + l;
#pragma unroll
            for (int i = 0; i < 8; i++) {
                const uint4 t = keep_in_l2 ? __ldg(p + 4 * i) : __ldcs(p + 4 * i);
                v[i][0] = t.x; v[i][1] = t.y; v[i][2] = t.z; v[i][3] = t.w;
            }
        } else {
            const ulonglong2* p = reinterpret_cast<const ulonglong2*>(x) + 2 * l;
#pragma unroll
            for (int i = 0; i < 8; i++) {
                const ulonglong2 t0 = keep_in_l2 ? __ldg(p + 8 * i) : __ldcs(p + 8 * i);
                const ulonglong2 t1 = keep_in_l2 ? __ldg(p + 8 * i + 1) : __ldcs(p + 8 * i + 1);
                v[i][0] = t0.x; v[i][1] = t0.y; v[i][2] = t1.x; v[i][3] = t1.y;
            }
        }
    } else {                                         // ragged / unaligned / missing blocks: guarded scalar loads
#pragma unroll
        for (int i = 0; i < 8; i++)
#pragma unroll
            for (int c = 0; c < 4; c++) {
                const int j = 16 * i + 4 * l + c;
                v[i][c] = (j < m) ? x[j] : (T)0;
            }
    }
}

// ---- E1: deltas, d_0 = 0, zero beyond m. One shuffle per row step:
// a lane needs the last ID of the previous row, which lives in lane-1 (same step) or, for l = 0,
// in lane+3 (previous step) — lane l = 3 publishes its previous step's value for that purpose.
template <int W>
__device__ __forceinline__ void quad_deltas(const typename IdT<W>::T (&v)[8][4], int m,
                                            typename IdT<W>::T (&d)[8][4]) {
    using T = typename IdT<W>::T;
    const int lane = threadIdx.x & 31, l = lane & 3;
    const int src = (l == 0) ? lane + 3 : lane - 1;
#pragma unroll
    for (int i = 0; i < 8; i++) {
        const T pub = (l == 3 && i > 0) ? v[i - 1][3] : v[i][3];
        T prev = __shfl_sync(kFull, pub, src);
        if (i == 0 && l == 0) prev = v[0][0];
        d[i][0] = v[i][0] - prev;
        d[i][1] = v[i][1] - v[i][0];
        d[i][2] = v[i][2] - v[i][1];
        d[i][3] = v[i][3] - v[i][2];
    }
    if (!__all_sync(kFull, m == kBlk)) {
#pragma unroll
        for (int i = 0; i < 8; i++)
#pragma unroll
            for (int c = 0; c < 4; c++)
                if (16 * i + 4 * l + c >= m) d[i][c] = 0;
    }
}

// quad-wide reductions (lanes 4q..4q+3)
__device__ __forceinline__ uint32_t quad_or(uint32_t x) {
    x |= __shfl_xor_sync(kFull, x, 1);
    return x | __shfl_xor_sync(kFull, x, 2);
}
__device__ __forceinline__ uint32_t quad_add(uint32_t x) {
    x += __shfl_xor_sync(kFull, x, 1);
    return x + __shfl_xor_sync(kFull, x, 2);
}
__device__ __forceinline__ uint32_t quad_min(uint32_t x) {
    x = min(x, __shfl_xor_sync(kFull, x, 1));
    return min(x, __shfl_xor_sync(kFull, x, 2));
}
__device__ __forceinline__ uint32_t quad_max(uint32_t x) {
    x = max(x, __shfl_xor_sync(kFull, x, 1));
    return max(x, __shfl_xor_sync(kFull, x, 2));
}

// ---- E2: canonical b of the quad's block (FORMAT.md §2: exact argmin of the block size over
// b in 0..maxw, ties to the largest b). Same window argument as choose_b in block_encode.cuh:
// the 9 candidates [top-8, top] are costed from nibble counters (pattern 0x11111111 << 4t marks the
// thresholds at which a value of width top-t is an exception); the chain of windows stops when
// the exceptions above the window alone cost at least the best size, and jumps over widths no
// value has. Returns key = size << 14 | (64 - b) << 7 | n_exc in every lane of the quad.
template <int W, typename DT>
__device__ __forceinline__ uint32_t quad_choose_b(const DT (&d)[8][4]) {
    const int l = quad_l();
    constexpr int kBits = 8 * (int)sizeof(DT);
    int top;
    {
        DT o = 0;
#pragma unroll
        for (int i = 0; i < 8; i++) o |= d[i][0] | d[i][1] | d[i][2] | d[i][3];
        uint32_t lo = (uint32_t)o, hi = 0;
        if constexpr (sizeof(DT) == 8) hi = (uint32_t)(o >> 32);
        lo = quad_or(lo);
        if constexpr (sizeof(DT) == 8) hi = quad_or(hi);
        top = hi ? 64 - __clz(hi) : 32 - __clz(lo);
    }
    uint32_t cnt_above = 0, best = 0xffffffffu;
    bool active = true;
    while (true) {
        uint32_t acc[3] = {0u, 0u, 0u};
        const int off = top - kBits;                 // t = top - width = clz + off
#pragma unroll
        for (int i = 0; i < 8; i++)
#pragma unroll
            for (int c = 0; c < 4; c++) {
                int clz;
                if constexpr (sizeof(DT) == 8) clz = __clzll(d[i][c]); else clz = __clz(d[i][c]);
                acc[i / 3] += shl32(0x11111111u, (uint32_t)(4 * (clz + off)));   // t < 0 or t >= 8: shift clamps to 0
            }
        uint32_t lo = (acc[0] & 0x0f0f0f0fu) + (acc[1] & 0x0f0f0f0fu) + (acc[2] & 0x0f0f0f0fu);
        uint32_t hi = ((acc[0] >> 4) & 0x0f0f0f0fu) + ((acc[1] >> 4) & 0x0f0f0f0fu) + ((acc[2] >> 4) & 0x0f0f0f0fu);
        lo = quad_add(lo);                           // bytes: exceptions added at s = 1,3,5,7 (b = top - s)
        hi = quad_add(hi);                           //                            s = 2,4,6,8
        uint32_t key = 0xffffffffu;
#pragma unroll
        for (int u = 0; u < 3; u++) {
            const int s = l + 4 * u;                 // this lane's candidates: s = l, l+4, l+8
            if (s <= 8 && s <= top && active) {
                uint32_t n = cnt_above;
                if (s > 0) n += ((((s - 1) & 1) ? hi : lo) >> (8 * ((s - 1) >> 1))) & 0xffu;
                const uint32_t b = (uint32_t)(top - s);
                key = min(key, ((16u + 16u * b + exc_bytes<W>(n)) << 14) | ((64u - b) << 7) | n);
            }
        }
        best = min(best, quad_min(key));
        const uint32_t n_bot = cnt_above + ((hi >> 24) & 0xffu);       // exceptions at b = top - 8
        active = active && top > 8 && (16u + exc_bytes<W>(n_bot)) < (best >> 14);
        if (!__any_sync(kFull, active)) break;
        uint32_t below = 0;                          // widest value not above top - 8
#pragma unroll
        for (int i = 0; i < 8; i++)
#pragma unroll
            for (int c = 0; c < 4; c++) {
                const uint32_t w = (uint32_t)bitlen<DT>(d[i][c]);
                below = max(below, (int)w <= top - 8 ? w : 0u);
            }
        below = quad_max(below);
        if (active) { top = (int)below; cnt_above = n_bot; }
    }
    return best;
}


// ---- E4: staging -----------------------------------------------------------------------
// Per-warp shared memory: the batch's masked values (row-major per block, padded stride) and the
// batch's assembled blocks (header | payload | exceptions), canonical size <= 16 + 16 W each.
template <int W>
struct QuadStage {
    static constexpr int kOutStride = 16 + 16 * W;              // bytes; /4 == 4 (mod 32) words
    static constexpr int kValWords = kValStride * (W / 32);     // u64 values take two words
    alignas(16) uint32_t vals[kQuadBlocks * kValWords];
    alignas(16) unsigned char out[kQuadBlocks * kOutStride];
};

// masked low parts of the quad's rows -> vals (row owner, 128-bit stores)
template <typename DT>
__device__ __forceinline__ void quad_stage_vals(uint32_t* __restrict__ vq, const DT (&d)[8][4], uint32_t b) {
    const int l = quad_l();
    if constexpr (sizeof(DT) == 4) {
        const uint32_t mask = b >= 32 ? 0xffffffffu : ((1u << b) - 1u);
#pragma unroll
        for (int i = 0; i < 8; i++)
            reinterpret_cast<uint4*>(vq)[4 * i + l] =
                make_uint4(d[i][0] & mask, d[i][1] & mask, d[i][2] & mask, d[i][3] & mask);
    } else {
        const uint64_t mask = b >= 64 ? ~0ull : ((1ull << b) - 1ull);
#pragma unroll
        for (int i = 0; i < 8; i++) {
            ulonglong2* p = reinterpret_cast<ulonglong2*>(vq) + 2 * (4 * i + l);
            p[0] = make_ulonglong2(d[i][0] & mask, d[i][1] & mask);
            p[1] = make_ulonglong2(d[i][2] & mask, d[i][3] & mask);
        }
    }
}

// Exceptions of the quad's block (n_exc > 0): positions ascending + high parts, FORMAT.md §2.
// The quad builds the block's 128-bit exception bitmap, parks the high parts in the (not yet
// used) vals area, then walks the bitmap: exception number e is written by lane e mod 4.
// Must be called by the whole warp (contains __syncwarp); quads with n_exc == 0 idle through it.
template <int W, typename DT>
__device__ __forceinline__ void quad_exceptions(uint32_t* __restrict__ vq, unsigned char* __restrict__ oq,
                                                const DT (&d)[8][4], uint32_t b, uint32_t n_exc) {
    using T = typename IdT<W>::T;
    constexpr uint32_t E = W / 8;
    const int l = quad_l();
    const bool on = n_exc > 0;
    uint32_t bm[4] = {0u, 0u, 0u, 0u};
    if (on) {
#pragma unroll
        for (int i = 0; i < 8; i++) {
            DT h[4];
#pragma unroll
            for (int c = 0; c < 4; c++) {
                h[c] = shr_clamp<DT>(d[i][c], b);
                if (h[c] != 0) bm[i >> 1] |= 1u << (16 * (i & 1) + 4 * l + c);   // j = 16 i + 4 l + c
            }
            if constexpr (sizeof(DT) == 4) {
                reinterpret_cast<uint4*>(vq)[4 * i + l] = make_uint4(h[0], h[1], h[2], h[3]);
            } else {
                ulonglong2* p = reinterpret_cast<ulonglong2*>(vq) + 2 * (4 * i + l);
                p[0] = make_ulonglong2(h[0], h[1]);
                p[1] = make_ulonglong2(h[2], h[3]);
            }
        }
        unsigned char* e = oq + 16 + 16 * b;                     // zero the area: pads must be 0
        const uint32_t eb = exc_bytes<W>(n_exc);
        for (uint32_t x = l; x < eb / 16; x += 4) reinterpret_cast<uint4*>(e)[x] = make_uint4(0, 0, 0, 0);
    }
#pragma unroll
    for (int w = 0; w < 4; w++) bm[w] = quad_or(bm[w]);
    __syncwarp();
    if (on) {
        unsigned char* e = oq + 16 + 16 * b;
        T* high = reinterpret_cast<T*>(e + ((n_exc + E - 1) & ~(E - 1)));
        const DT* hv = reinterpret_cast<const DT*>(vq);
        uint32_t rank = 0;
#pragma unroll
        for (int w = 0; w < 4; w++) {
            uint32_t mk = bm[w];
            while (mk) {
                const uint32_t p = 32u * w + (uint32_t)__ffs(mk) - 1u;
                mk &= mk - 1u;
                if ((rank & 3u) == (uint32_t)l) {
                    e[rank] = (unsigned char)p;
                    high[rank] = (T)hv[p];
                }
                rank++;
            }
        }
    }
    __syncwarp();
}

// One column of the payload, packed sequentially by its owner lane (b <= 32, 32-bit values).
// For b <= 16 (<= 8) neighbouring rows are first merged into 2b- (4b-) bit items with one IMAD each,
// which halves (quarters) the length of the sequential part.
#define BFSC_EMIT_ITEM(xv)                                               \
    {                                                                    \
        const uint32_t x_ = (xv);                                        \
        acc |= x_ << have;                                               \
        uint32_t nh = have + bw;                                         \
        if (nh >= 32u) {                                                 \
            *outp = acc;                                                 \
            outp += 4;                                                   \
            acc = shr32(x_, 32u - have);                                 \
            nh -= 32u;                                                   \
        }                                                                \
        have = nh;                                                       \
    }

__device__ __forceinline__ void quad_pack_column32(const uint32_t* __restrict__ col /* row r at col[4r] */,
                                                   uint32_t* __restrict__ outp /* word k at outp[4k] */, uint32_t b) {
    if (b == 0) return;
    uint32_t u[32];
#pragma unroll
    for (int r = 0; r < 32; r++) u[r] = col[4 * r];
    uint32_t acc = 0, have = 0;
    if (b <= 8) {
        const uint32_t m1 = 1u << b, m2 = 1u << (2 * b), bw = 4 * b;
#pragma unroll
        for (int p = 0; p < 8; p++) {
            const uint32_t a0 = u[4 * p] + u[4 * p + 1] * m1, a1 = u[4 * p + 2] + u[4 * p + 3] * m1;
            BFSC_EMIT_ITEM(a0 + a1 * m2)
        }
    } else if (b <= 16) {
        const uint32_t m1 = 1u << b, bw = 2 * b;
#pragma unroll
        for (int p = 0; p < 16; p++) BFSC_EMIT_ITEM(u[2 * p] + u[2 * p + 1] * m1)
    } else {
        const uint32_t bw = b;
#pragma unroll
        for (int r = 0; r < 32; r++) BFSC_EMIT_ITEM(u[r])
    }
}
#undef BFSC_EMIT_ITEM

// Wide values (u64 deltas, any b <= 64): plain sequential packer with a 128-bit window.
__device__ __forceinline__ void quad_pack_column64(const uint64_t* __restrict__ col /* row r at col[4r] */,
                                                   uint32_t* __restrict__ outp, uint32_t b) {
    if (b == 0) return;
    uint64_t lo = 0, hi = 0;
    uint32_t have = 0;
    for (int r = 0; r < 32; r++) {
        const uint64_t x = col[4 * r];
        lo |= shl64(x, have);
        hi |= have ? shr64(x, 64u - have) : 0ull;     // have < 32 here
        have += b;
        while (have >= 32u) {
            *outp = (uint32_t)lo;
            outp += 4;
            lo = (lo >> 32) | (hi << 32);
            hi >>= 32;
            have -= 32u;
        }
    }
}

}  // namespace bfsc
