// quad_encode.cuh — encode steps E1, E2, E4 with FOUR LANES PER BLOCK: a warp works on 8
// consecutive 128-ID blocks at once ("batch"). lane = 4*q + l: q = block of the batch, l = lane
// of the quad. Per-block scalar work (sizes, offsets, headers) then costs 1/8 of a warp
// instruction per block instead of a whole one, and nothing needs a full-warp reduction.
//
// Ownership of a block's 128 values (j = 4r + c, row r = 0..31, column c = 0..3): lane c of the quad is the
// COLUMN OWNER of column c. The raw IDs are staged in shared memory by cp.async; lane c forms the 32 deltas of
// its column there (E1), counts widths (E2) and packs the column's bit stream (E4, FORMAT.md payload)
// sequentially from registers — the values never change hands between E1 and E4.
#pragma once
#include "common.cuh"

namespace bfsc {

constexpr int kQuadBlocks = 8;                       // blocks per warp batch
__device__ __forceinline__ int quad_l() { return threadIdx.x & 3; }

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
// b in 0..maxw, ties to the largest b). Window argument:
// the 9 candidates [top-8, top] are costed from nibble counters (pattern 0x11111111 << 4t marks the
// thresholds at which a value of width top-t is an exception); the chain of windows stops when
// the exceptions above the window alone cost at least the best size, and jumps over widths no
// value has. Returns key = size << 14 | (64 - b) << 7 | n_exc in every lane of the quad.
// Position of the most significant set bit (0xffffffff for 0). volatile: the widths are recomputed in
// every window instead of being kept in 32 registers across the window loop.
__device__ __forceinline__ uint32_t msb_pos(uint32_t x) {
    uint32_t r;
    asm volatile("bfind.u32 %0, %1;" : "=r"(r) : "r"(x));
    return r;
}

// a * b + c as ONE IMAD (fma pipe): the alu pipe (LOP3 / SHF / IADD3, one warp instruction per two cycles
// and scheduler) is the busiest unit of the encoder.
__device__ __forceinline__ uint32_t mad_fma_pipe(uint32_t a, uint32_t b, uint32_t c) {
    uint32_t r;
    asm("mad.lo.u32 %0, %1, %2, %3;" : "=r"(r) : "r"(a), "r"(b), "r"(c));
    return r;
}

template <int W>
__device__ __forceinline__ uint32_t quad_choose_b(const uint32_t (&d)[32]) {
    const int l = quad_l();
    int top;
    {
        uint32_t o = 0;
#pragma unroll
        for (int i = 0; i < 32; i++) o |= d[i];
        top = 32 - __clz(quad_or(o));
    }
    uint32_t cnt_above = 0, best = 0xffffffffu;
    bool active = true;
    while (true) {
        uint32_t acc[3] = {0u, 0u, 0u};
        const int K = 4 * (top - 1);                 // t = top - width = (top - 1) - msb_pos; msb_pos(0) = -1
#pragma unroll
        for (int i = 0; i < 32; i++)                 // t < 0 or t >= 8: the shift clamps to 0
            acc[i / 12] = mad_fma_pipe(shl32(1u, (uint32_t)(K - 4 * (int)msb_pos(d[i]))), 0x11111111u, acc[i / 12]);
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
        // Next window: [top - 16, top - 8] (its first candidate is this window's last: evaluated twice, harmless). The
        // widths no value has are not skipped: finding the widest value below the window costs a pass over the 32
        // values of its own (3 instructions each), as much as three quarters of a window.
        if (active) { top -= 8; cnt_above = n_bot; }
    }
    return best;
}

// ---- E2 of the no-exception codec (FORMAT.md §7, mode 2 = BP128-D1; the thesis's codec class S4-BP128,
// PAPER.md L1052-1056): b = width of the block's widest delta (eq. 6), n_exc = 0. Same key layout.
__device__ __forceinline__ uint32_t quad_max_width_key(const uint32_t (&d)[32]) {
    uint32_t o = 0;
#pragma unroll
    for (int i = 0; i < 32; i++) o |= d[i];
    const uint32_t top = 32u - (uint32_t)__clz(quad_or(o));
    return ((16u + 16u * top) << 14) | ((64u - top) << 7);
}

// ---- E4: staging geometry ----------------------------------------------------------------
// Per warp: a staging area (the batch's 128 deltas per block, row-major) and an image area (the
// assembled block: header | payload | exceptions). Both hold 8 slots of 33 16-byte chunks; slot q
// starts at chunk 33 q + 3 ((q + 1) >> 1) = {0,36,69,105,138,174,207,243}: the residues mod 8 are
// {0,4,5,1,2,6,7,3}, so that (i) the 8 quads' column reads/writes (32-bit, same row) hit 8 distinct
// 16-byte bank groups and (ii) the two quads of a 128-bit phase (2h, 2h+1) are 4 groups apart —
// row-owner 128-bit accesses are conflict-free too.
constexpr int kSlotChunks = 33;
constexpr int kAreaChunks = 243 + kSlotChunks;                  // 276 chunks = 4416 B
__device__ __forceinline__ int quad_slot_chunk(int q) { return 33 * q + 3 * ((q + 1) >> 1); }

// One column of the payload (FORMAT.md §2 "Payload"), packed sequentially by its owner lane from
// registers: row r's low b bits at stream bits [r b, (r+1) b); word k goes to outp[4k].
// For b <= 8 (<= 16) four (two) neighbouring rows are first merged into one item with IMADs, which
// quarters (halves) the sequential part. b in 1..32.
#define BFSC_EMIT_ITEM(xv)                                               \
    {                                                                    \
        const uint32_t x_ = (xv);                                        \
        acc |= x_ << have;                                               \
        const uint32_t hi_ = __funnelshift_l(x_, 0u, have);              \
        const uint32_t nh_ = have + bw;                                  \
        if (nh_ >= 32u) {                                                \
            *outp = acc;                                                 \
            outp += 4;                                                   \
            acc = hi_;                                                   \
        }                                                                \
        have = nh_ & 31u;                                                \
    }

__device__ __forceinline__ void col_pack32(const uint32_t (&u)[32], uint32_t b, uint32_t* __restrict__ outp) {
    const uint32_t mask = 0xffffffffu >> (32u - b);
    uint32_t acc = 0, have = 0;
    if (b <= 8) {
        const uint32_t m1 = 1u << b, m2 = 1u << (2 * b), bw = 4 * b;
#pragma unroll
        for (int p = 0; p < 8; p++) {
            const uint32_t a0 = (u[4 * p] & mask) + (u[4 * p + 1] & mask) * m1;
            const uint32_t a1 = (u[4 * p + 2] & mask) + (u[4 * p + 3] & mask) * m1;
            BFSC_EMIT_ITEM(a0 + a1 * m2)
        }
    } else if (b <= 16) {
        const uint32_t m1 = 1u << b, bw = 2 * b;
#pragma unroll
        for (int p = 0; p < 16; p++) BFSC_EMIT_ITEM((u[2 * p] & mask) + (u[2 * p + 1] & mask) * m1)
    } else {
        const uint32_t bw = b;
#pragma unroll
        for (int r = 0; r < 32; r++) BFSC_EMIT_ITEM(u[r] & mask)
    }
}
#undef BFSC_EMIT_ITEM

// ---- E1 (column owner): raw IDs staged by cp.async, deltas computed by the lane that packs them ----
// The quad's block is copied global -> shared as ALIGNED 16-byte chunks (cp.async.cg, no registers,
// any element alignment: the block's first ID sits e elements into chunk 0). A slot holds
// kSlotChunks (u32) / 2 kSlotChunks (u64) chunks; u64 slots are dense (66 q: the residues mod 8 of
// a 16-lane phase's four quads are {0,2,4,6}), u32 slots use quad_slot_chunk.
template <int W> __device__ __forceinline__ int raw_slot_chunk(int q) {
    if constexpr (W == 32) return quad_slot_chunk(q); else return 2 * kSlotChunks * q;
}
template <int W> struct RawCfg { static constexpr int kAreaChunks = (W == 32) ? bfsc::kAreaChunks : 16 * kSlotChunks; };

__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gmem_src) {
    const uint32_t d = (uint32_t)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(d), "l"(gmem_src) : "memory");
}
// Same, reading only the first src_bytes (1..16) of the chunk; the rest of the 16 bytes is zero-filled.
__device__ __forceinline__ void cp_async16_part(void* smem_dst, const void* gmem_src, int src_bytes) {
    const uint32_t d = (uint32_t)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(d), "l"(gmem_src), "r"(src_bytes) : "memory");
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N> __device__ __forceinline__ void cp_async_wait_group() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }   // all but the newest N groups

// x = block's first ID (m valid IDs, m <= 0: nothing to copy). Lane l of the quad copies chunks l, l+4, ...
template <int W>
__device__ __forceinline__ void quad_prefetch(uint4* __restrict__ slot, const typename IdT<W>::T* __restrict__ x, int m) {
    using T = typename IdT<W>::T;
    constexpr int EPC = 16 / (int)sizeof(T);                    // elements per chunk
    constexpr int kRounds = kBlk / EPC / 4;                      // 8 (u32) / 16 (u64) full rounds, + 1 for e > 0
    if (m <= 0) return;
    const int l = quad_l();
    const uintptr_t addr = reinterpret_cast<uintptr_t>(x);
    const int e = (int)(addr & 15) / (int)sizeof(T);
    const uint4* src = reinterpret_cast<const uint4*>(addr & ~(uintptr_t)15) + l;
    const int nchunk = (e + m + EPC - 1) / EPC;
    if (nchunk == kBlk / EPC) {
#pragma unroll
        for (int i = 0; i < kRounds; i++) cp_async16(slot + 4 * i + l, src + 4 * i);
    } else {                                                     // ragged block (the last one of its buffer), or e > 0:
        const int tail = (e + m) * (int)sizeof(T) - 16 * (nchunk - 1);   // nothing is read beyond the block's last ID
#pragma unroll
        for (int i = 0; i <= kRounds; i++)
            if (4 * i + l < nchunk) cp_async16_part(slot + 4 * i + l, src + 4 * i, 4 * i + l == nchunk - 1 ? tail : 16);
    }
}

// Column owner c: d[r] = delta of ID j = 4r + c (d_0 = 0, 0 beyond m), from the staged
// raw IDs. Returns the block's first ID (valid in lane c = 0) and, for u64, whether some delta of
// the lane does not fit 32 bits.
template <int W>
__device__ __forceinline__ typename IdT<W>::T col_deltas(const typename IdT<W>::T* __restrict__ raw /* slot + e */, int m,
                                                         uint32_t (&d)[32], bool& wide_lane) {
    using T = typename IdT<W>::T;
    const int c = quad_l();
    const T* p = raw + c;
    T first = p[0];
    uint32_t hi_or = 0;
#pragma unroll
    for (int r = 0; r < 32; r++) {
        const T cur = (r == 0) ? first : p[4 * r];
        const T prev = (r == 0) ? p[c == 0 ? 0 : -1] : p[4 * r - 1];
        const T dd = cur - prev;
        d[r] = (uint32_t)dd;
        if constexpr (W == 64) hi_or |= (uint32_t)(dd >> 32);
    }
    if (!__all_sync(kFull, m == kBlk)) {
        hi_or = 0;
#pragma unroll
        for (int r = 0; r < 32; r++) {
            if (4 * r + c >= m) d[r] = 0;
            if constexpr (W == 64) { if (4 * r + c < m && r > 0) hi_or |= (uint32_t)((p[4 * r] - p[4 * r - 1]) >> 32); }
        }
        if constexpr (W == 64) { if (c > 0 && c < m) hi_or |= (uint32_t)((p[0] - p[-1]) >> 32); }
    }
    wide_lane = hi_or != 0;
    return first;
}


// Exceptions of the quad's block (FORMAT.md §2 "Exceptions"), column owner, 32-bit deltas (for W = 64 the high
// parts are zero-extended). e = image + 16 + 16 b. Exception number `rank` (ascending position j = 4r + c) is
// written by the lane that owns it: each lane builds the 32-bit mask of its own exceptions (bit r), the quad
// exchanges the four masks, and rank = number of exceptions in earlier rows plus those of lower columns in the
// same row. The high part is recomputed from the staged RAW IDs.
// Must be called by the whole warp (shuffles, __syncwarp); quads with n_exc == 0 idle through it.
template <int W>
__device__ __forceinline__ void col_exceptions_raw(const uint32_t (&u)[32], const typename IdT<W>::T* __restrict__ raw,
                                                   unsigned char* __restrict__ e, uint32_t b, uint32_t n_exc) {
    using T = typename IdT<W>::T;
    constexpr uint32_t E = W / 8;
    const int lane = threadIdx.x & 31, c = lane & 3;
    const bool on = n_exc > 0;                               // then b < 32
    uint32_t mk = 0;
    if (on) {
        const uint32_t mask = (1u << b) - 1u;
#pragma unroll
        for (int r = 0; r < 32; r++)
            if (u[r] > mask) mk |= 1u << r;
        const uint32_t eb = exc_bytes<W>(n_exc);             // zero the area: pads must be 0
        for (uint32_t x = c; x < eb / 16; x += 4) reinterpret_cast<uint4*>(e)[x] = make_uint4(0, 0, 0, 0);
    }
    const uint32_t M0 = __shfl_sync(kFull, mk, (lane & ~3) + 0), M1 = __shfl_sync(kFull, mk, (lane & ~3) + 1);
    const uint32_t M2 = __shfl_sync(kFull, mk, (lane & ~3) + 2), M3 = __shfl_sync(kFull, mk, (lane & ~3) + 3);
    __syncwarp();
    if (on) {
        T* high = reinterpret_cast<T*>(e + ((n_exc + E - 1) & ~(E - 1)));
        uint32_t rest = mk;
        while (rest) {
            const uint32_t r = (uint32_t)__ffs(rest) - 1u;
            rest &= rest - 1u;
            const uint32_t below = (1u << r) - 1u, incl = (2u << r) - 1u;
            const uint32_t rank = __popc(M0 & (c > 0 ? incl : below)) + __popc(M1 & (c > 1 ? incl : below)) +
                                  __popc(M2 & (c > 2 ? incl : below)) + __popc(M3 & below);
            const uint32_t pos = 4u * r + (uint32_t)c;       // > 0: d_0 = 0 is never an exception
            e[rank] = (unsigned char)pos;
            high[rank] = (T)(raw[pos] - raw[pos - 1]) >> b;
        }
    }
    __syncwarp();
}

}  // namespace bfsc
