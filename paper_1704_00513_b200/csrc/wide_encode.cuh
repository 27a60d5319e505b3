// wide_encode.cuh — slow paths of the encoder, for the blocks the fast path does not take:
//   * u64 warp batches in which some delta does not fit 32 bits (b may exceed 32, a packed value may
//     span three words). Never the case for sorted vertex IDs below 2^32 (every BASELINE config);
//     they exist so that ANY u64 input round-trips (FORMAT.md §2: modular deltas);
//   * blocks whose image does not fit the fast path's 256-byte shared-memory slot (b >= 15 or so:
//     nearly incompressible data).
// Both assemble the block straight into global memory once its offset is known.
#pragma once
#include "common.cuh"

namespace bfsc {

// Whole warp calls; lane = 4q + l. x: the quad's block (first ID, re-read from global memory), m valid
// IDs, key = size<<14 | (64-b)<<7 | n_exc, dst = final address of the block or nullptr (nothing to do
// for this quad). No shared memory: lane l packs column l from global memory, lane 0 lists the exceptions.
template <int W>
__device__ __noinline__ void late_emit(const typename IdT<W>::T* __restrict__ x, int m, uint32_t key,
                                       unsigned char* __restrict__ dst) {
    using T = typename IdT<W>::T;
    constexpr uint32_t E = W / 8;
    const int l = threadIdx.x & 3;
    const uint32_t b = 64u - ((key >> 7) & 127u), n_exc = key & 127u;
    if (dst == nullptr || m <= 0) return;
    auto delta = [&](int j) -> uint64_t { return (j > 0 && j < m) ? (uint64_t)(T)(x[j] - x[j - 1]) : 0ull; };   // E1 (L979-986)
    if (b > 0) {                                                             // E4: column l
        const uint64_t mask = b >= 64 ? ~0ull : ((1ull << b) - 1ull);
        uint32_t* outp = reinterpret_cast<uint32_t*>(dst + 16) + l;
        uint64_t lo = 0, hi = 0;
        uint32_t have = 0;
        for (int r = 0; r < 32; r++) {
            const uint64_t v = delta(4 * r + l) & mask;
            lo |= shl64(v, have);
            hi |= have ? shr64(v, 64u - have) : 0ull;                        // have < 32 here
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
    if (l == 0) {
        reinterpret_cast<unsigned long long*>(dst)[0] = (unsigned long long)x[0];
        reinterpret_cast<unsigned long long*>(dst)[1] = (unsigned long long)(b | (n_exc << 8));
        if (n_exc > 0) {                                                     // then b < W
            unsigned char* e = dst + 16 + 16 * b;
            const uint32_t eb = exc_bytes<W>(n_exc);
            for (uint32_t t = 0; t < eb / 16; t++) reinterpret_cast<uint4*>(e)[t] = make_uint4(0, 0, 0, 0);
            T* high = reinterpret_cast<T*>(e + ((n_exc + E - 1) & ~(E - 1)));
            uint32_t rank = 0;
            for (int j = 0; j < kBlk; j++) {
                const uint64_t hv = delta(j) >> b;
                if (hv) { e[rank] = (unsigned char)j; high[rank] = (T)hv; rank++; }
            }
        }
    }
}

// E2 for a warp batch with wide deltas: exact argmin of the block size over b in 0..maxw, ties to
// the largest b (FORMAT.md §2), from a 65-bin histogram of the widths in shared memory. Whole warp
// calls; raw = the quad's staged IDs (block's first ID at raw[0]); hist = 65 words of scratch per quad.
// no_exc: the BP128 rule (FORMAT.md §7): b = maxw, n_exc = 0.
__device__ __noinline__ uint32_t wide_choose_b(const uint64_t* __restrict__ raw, int m, uint32_t* __restrict__ hist,
                                               bool no_exc) {
    const int lane = threadIdx.x & 31, l = lane & 3;
    for (int k = l; k < 65; k += 4) hist[k] = 0;
    __syncwarp();
    for (int j = l; j < kBlk; j += 4) {
        const uint64_t d = (j > 0 && j < m) ? raw[j] - raw[j - 1] : 0ull;
        atomicAdd(&hist[64 - __clzll((long long)d)], 1u);
    }
    __syncwarp();
    uint32_t best = 0xffffffffu;
    if (l == 0) {
        int maxw = 64;
        while (maxw > 0 && hist[maxw] == 0) maxw--;
        uint32_t n = 0;
        for (int b = maxw; b >= (no_exc ? maxw : 0); b--) {      // descending: a tie keeps the larger b
            const uint32_t key = ((16u + 16u * (uint32_t)b + exc_bytes<64>(n)) << 14) | ((64u - (uint32_t)b) << 7) | n;
            if ((key >> 14) < (best >> 14)) best = key;
            n += hist[b];
        }
    }
    __syncwarp();
    return __shfl_sync(kFull, best, lane & ~3);
}

}  // namespace bfsc
