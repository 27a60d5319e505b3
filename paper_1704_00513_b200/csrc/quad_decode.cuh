// quad_decode.cuh — decode steps D1-D4 with FOUR LANES PER BLOCK: a warp decodes 8 consecutive
// 128-ID blocks at once. lane = 4*q + l: q = block of the batch, l = lane of the quad.
// Lane l owns rows r = 4i + l, i = 0..7 (IDs 16i + 4l .. 16i + 4l + 3): per step i the quad writes
// 64 (u32) / 128 (u64) contiguous bytes, so loads and stores are coalesced 128-bit accesses, and the
// per-block scalar work (header, directory, validation) costs 1/8 of a warp instruction per block.
//
// Fast path only: blocks of at most kDecSlotChunks - 2 16-byte chunks (b <= 16 without exceptions),
// staged in shared memory by cp.async. Larger blocks take the warp-per-block path of block_decode.cuh.
#pragma once
#include "common.cuh"

namespace bfsc {

constexpr int kDecBlocks = 8;                 // blocks per warp batch
constexpr int kDecSpanMax = 17;               // largest staged block, in 16-byte chunks (272 B)
constexpr int kDecSlotChunks = 19;            // slot stride: one chunk of slack for the unpack's second read; 19 q mod 8 distinct
constexpr int kDecStageChunks = kDecBlocks * kDecSlotChunks;

__device__ __forceinline__ void dec_cp_async16(void* smem_dst, const void* gmem_src) {
    const uint32_t d = (uint32_t)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(d), "l"(gmem_src) : "memory");
}
__device__ __forceinline__ void dec_cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }

// D1: stage the quad's block (span16 <= kDecSpanMax chunks at blk) into its slot; lane l copies chunks l, l+4, ...
__device__ __forceinline__ void quad_stage_block(uint4* __restrict__ slot, const unsigned char* __restrict__ blk,
                                                 uint32_t span16, int l) {
    const uint4* src = reinterpret_cast<const uint4*>(blk);
#pragma unroll
    for (int i = 0; i < (kDecSpanMax + 3) / 4; i++) {
        const uint32_t c = 4 * i + l;
        if (c < span16) dec_cp_async16(slot + c, src + c);
    }
}

// D2: low parts of the lane's rows from the staged payload P (b vectors of 128 bits, b <= 16; FORMAT.md §2
// "Payload"). Row r's values sit at bits [r b, r b + b) of each column stream; the second vector read may
// be one past the payload (slack chunk / exception area): its bits are masked off.
__device__ __forceinline__ void quad_unpack(const uint4* __restrict__ P, uint32_t b, int l, uint32_t (&d)[8][4]) {
    const uint32_t mask = (1u << b) - 1u;
    uint32_t bit = (uint32_t)l * b;
#pragma unroll
    for (int i = 0; i < 8; i++) {
        const uint32_t k0 = bit >> 5, sh = bit & 31u;
        const uint4 lo = P[k0], hi = P[k0 + 1];
        d[i][0] = __funnelshift_r(lo.x, hi.x, sh) & mask;
        d[i][1] = __funnelshift_r(lo.y, hi.y, sh) & mask;
        d[i][2] = __funnelshift_r(lo.z, hi.z, sh) & mask;
        d[i][3] = __funnelshift_r(lo.w, hi.w, sh) & mask;
        bit += 4u * b;
    }
}

// D3: exceptions through a per-warp patch table (128 entries per block, all zero between uses): the quad
// scatters high << b at each position, every lane ORs its rows' entries in, the scattering lanes clear
// them again. e = staged exception area. Returns false on a malformed position. Whole warp calls;
// quads with n_exc == 0 idle through it (their table entries are zero: tab is still read).
template <int W>
__device__ __forceinline__ bool quad_patch(typename IdT<W>::T* __restrict__ tab /* the quad's 128 entries */,
                                           const unsigned char* __restrict__ e, uint32_t b, uint32_t n_exc, int l,
                                           typename IdT<W>::T (&hi)[8][4]) {
    using T = typename IdT<W>::T;
    constexpr uint32_t E = W / 8;
    const T* high = reinterpret_cast<const T*>(e + ((n_exc + E - 1) & ~(E - 1)));
    bool ok = true;
    for (uint32_t x = l; x < n_exc; x += 4) {
        const uint32_t pos = e[x];
        if (pos >= (uint32_t)kBlk) ok = false; else tab[pos] = high[x] << b;
    }
    __syncwarp();
#pragma unroll
    for (int i = 0; i < 8; i++) {
        if constexpr (W == 32) {
            const uint4 t = reinterpret_cast<const uint4*>(tab)[4 * i + l];
            hi[i][0] = t.x; hi[i][1] = t.y; hi[i][2] = t.z; hi[i][3] = t.w;
        } else {
            const ulonglong2 t0 = reinterpret_cast<const ulonglong2*>(tab)[2 * (4 * i + l)];
            const ulonglong2 t1 = reinterpret_cast<const ulonglong2*>(tab)[2 * (4 * i + l) + 1];
            hi[i][0] = t0.x; hi[i][1] = t0.y; hi[i][2] = t1.x; hi[i][3] = t1.y;
        }
    }
    __syncwarp();
    for (uint32_t x = l; x < n_exc; x += 4) {
        const uint32_t pos = e[x];
        if (pos < (uint32_t)kBlk) tab[pos] = 0;
    }
    return ok;
}

// D4: inclusive scan of the block's 128 deltas + base (mod 2^W) and store of the first m IDs.
// v[i][c] = delta of ID 16i + 4l + c. Order of the IDs: i major, then lane, then c.
template <int W>
__device__ __forceinline__ void quad_scan_store(typename IdT<W>::T (&v)[8][4], typename IdT<W>::T base,
                                                typename IdT<W>::T* __restrict__ x, int m, int l) {
    using T = typename IdT<W>::T;
    T carry = base;
#pragma unroll
    for (int i = 0; i < 8; i++) {
        v[i][1] += v[i][0]; v[i][2] += v[i][1]; v[i][3] += v[i][2];      // prefix inside the row
        T inc = v[i][3];                                                 // inclusive scan of the row sums over the quad
        T t = __shfl_up_sync(kFull, inc, 1, 4);
        if (l >= 1) inc += t;
        t = __shfl_up_sync(kFull, inc, 2, 4);
        if (l >= 2) inc += t;
        const T tot = __shfl_sync(kFull, inc, 3, 4);
        const T off = carry + (inc - v[i][3]);
        v[i][0] += off; v[i][1] += off; v[i][2] += off; v[i][3] += off;
        carry += tot;
    }
    const bool vec_ok = (m == kBlk) && ((reinterpret_cast<uintptr_t>(x) & 15) == 0);
    if (__all_sync(kFull, vec_ok || m <= 0)) {
        if (m > 0) {
#pragma unroll
            for (int i = 0; i < 8; i++) {
                if constexpr (W == 32) {
                    __stcs(reinterpret_cast<uint4*>(x) + 4 * i + l, make_uint4(v[i][0], v[i][1], v[i][2], v[i][3]));
                } else {
                    ulonglong2* p = reinterpret_cast<ulonglong2*>(x) + 2 * (4 * i + l);
                    __stcs(p, make_ulonglong2(v[i][0], v[i][1]));
                    __stcs(p + 1, make_ulonglong2(v[i][2], v[i][3]));
                }
            }
        }
    } else {
#pragma unroll
        for (int i = 0; i < 8; i++)
#pragma unroll
            for (int c = 0; c < 4; c++) {
                const int jx = 16 * i + 4 * l + c;
                if (jx < m) x[jx] = v[i][c];
            }
    }
}

}  // namespace bfsc
