// encode.cu — bfsc_compress / bfsc_compress_batch (steps E0-E5).
#include "quad_encode.cuh"

namespace bfsc {

struct EncArgs {
    const void* ids;
    const unsigned long long* in_off;   // n_buf+1 element offsets, or nullptr (single buffer of n_single IDs)
    unsigned long long n_single;
    uint32_t n_buf;
    unsigned long long thr;             // raw threshold in bytes
    unsigned char* out;
    unsigned long long out_cap;
    unsigned long long* out_off;        // n_buf+1 (batch) or nullptr
    unsigned long long* out_total;      // single: *d_out_bytes, or nullptr
    uint32_t* status;
    WsView ws;
};

__device__ __forceinline__ unsigned long long buf_start(const EncArgs& a, uint32_t i) {
    return a.in_off ? a.in_off[i] : 0ull;
}
__device__ __forceinline__ unsigned long long buf_count(const EncArgs& a, uint32_t i) {
    return a.in_off ? a.in_off[i + 1] - a.in_off[i] : a.n_single;
}

// ---- E0: plan. One CTA; per buffer: mode, block count, fixed bytes; exclusive prefixes. ----
template <int W>
__global__ void __launch_bounds__(1024) k_enc_plan(EncArgs a) {
    __shared__ Scan2 sm[33];
    __shared__ int bad;
    constexpr unsigned long long E = W / 8;
    constexpr unsigned long long kTile = 256;                   // = kTileR of the fused kernel
    if (threadIdx.x == 0) bad = 0;
    __syncthreads();
    Scan2 carry{0, 0};
    for (uint32_t i0 = 0; i0 < a.n_buf; i0 += blockDim.x) {
        const uint32_t i = i0 + threadIdx.x;
        Scan2 v{0, 0};
        if (i < a.n_buf) {
            if (a.in_off && a.in_off[i + 1] < a.in_off[i]) bad = 1;
            const unsigned long long n = buf_count(a, i);
            const bool raw = n * E < a.thr;                               // FORMAT.md §1 (L1311)
            const unsigned long long nb = raw ? 0ull : (n + kBlk - 1) / kBlk;
            v.a = nb;
            v.b = raw ? 32ull + ((n * E + 15ull) & ~15ull) : 32ull + ((4ull * (nb + 1) + 15ull) & ~15ull);
        }
        Scan2 tot;
        Scan2 ex = block_scan_excl2(v, &tot, sm);
        if (i < a.n_buf) {
            a.ws.blk_first[i] = carry.a + ex.a;
            a.ws.fixed_prefix[i] = carry.b + ex.b;
            a.ws.stream_start[i] = 0;
        }
        carry.a += tot.a; carry.b += tot.b;
    }
    __syncthreads();
    {                                                    // look-back states of the fused kernel start invalid
        unsigned long long nt = (carry.a + kTile - 1) / kTile;
        if (nt > a.ws.tile_cap) nt = a.ws.tile_cap;
        for (unsigned long long q = threadIdx.x; q < nt; q += blockDim.x) a.ws.tile_state[q] = 0;
    }
    if (threadIdx.x == 0) {
        a.ws.blk_first[a.n_buf] = carry.a;
        a.ws.fixed_prefix[a.n_buf] = carry.b;
        a.ws.stream_start[a.n_buf] = 0;
        a.ws.hdr->total_blocks = carry.a;
        a.ws.hdr->fixed_total = carry.b;
        a.ws.hdr->ticket = 0;
        a.ws.hdr->grand16 = 0;
        a.ws.hdr->total_out = carry.b;
        const bool ok = !bad && carry.a <= a.ws.blk_cap && (carry.a + kTile - 1) / kTile <= a.ws.tile_cap;
        a.ws.hdr->ok = ok ? 1u : 0u;
        if (!ok) set_status(a.status, BFSC_ERR_INVALID_ARG);
    }
}

// ---- E1-E4 fused: one pass over HBM -----------------------------------------------------
// A CTA pulls tiles of kTileR consecutive blocks (128 KB of u32 IDs) by ticket.
//   pass A  (E1+E2): deltas, widths and the canonical b of every block; sizes to shared memory.
//   scan    (E3): intra-tile exclusive scan of the sizes, tile aggregate published, decoupled
//           look-back over the (few hundred) tiles in flight -> device-wide exclusive scan.
//   pass B  (E1+E4): the blocks are read again — still in the 126 MB L2, so HBM is read once —
//           packed in shared memory and stored with 128-bit stores at their final offsets, with
//           their directory entries.
// Both passes use four lanes per block (quad_encode.cuh): a warp works on 8 blocks at a time.
template <int W> struct EncCfg { static constexpr int kWarps = (W == 32) ? 8 : 4; };
constexpr int kTileR = 256;              // blocks per tile

constexpr unsigned long long kFlagAgg = 1ull << 62, kFlagPre = 2ull << 62, kValMask = (1ull << 62) - 1;

__device__ __forceinline__ unsigned long long ld_volatile_u64(const unsigned long long* p) {
    unsigned long long v;
    asm volatile("ld.volatile.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_volatile_u64(unsigned long long* p, unsigned long long v) {
    asm volatile("st.volatile.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}

template <int W>
__global__ void __launch_bounds__(EncCfg<W>::kWarps * 32) k_enc_fused(EncArgs a) {
    using T = typename IdT<W>::T;
    constexpr int kWarps = EncCfg<W>::kWarps, kThreads = kWarps * 32;
    extern __shared__ __align__(16) unsigned char dyn_smem[];
    QuadStage<W>* stage_all = reinterpret_cast<QuadStage<W>*>(dyn_smem);
    __shared__ uint32_t s_key[kTileR];               // pass A result per block: size<<14 | (64-b)<<7 | n_exc
    __shared__ uint32_t s_excl[kTileR + 1];          // exclusive scan of sizes (16-B units) inside the tile
    __shared__ uint32_t s_buf[kTileR];               // buffer of each block
    __shared__ int s_m[kTileR];                      // valid IDs of each block (0 = no block)
    __shared__ unsigned long long s_xoff[kTileR];    // element offset of the block's first ID
    __shared__ unsigned long long s_tile;
    __shared__ unsigned long long s_lb_sum[kWarps];
    __shared__ int s_lb_hit[kWarps];

    if (!a.ws.hdr->ok) return;
    const unsigned long long total = a.ws.hdr->total_blocks;
    const unsigned long long n_tiles = (total + kTileR - 1) / kTileR;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, tid = threadIdx.x;
    const int q = lane >> 2, l = lane & 3;
    QuadStage<W>& st = stage_all[warp];
    const T* ids = reinterpret_cast<const T*>(a.ids);

    while (true) {
        if (tid == 0) s_tile = atomicAdd(&a.ws.hdr->ticket, 1u);
        __syncthreads();
        const unsigned long long t = s_tile;
        if (t >= n_tiles) break;
        const unsigned long long g0 = t * kTileR;

        for (int j = tid; j < kTileR; j += kThreads) {           // bookkeeping: block g0 + j
            const unsigned long long g = g0 + j;
            int m = 0; uint32_t i = 0; unsigned long long xoff = 0;
            if (g < total) {
                i = find_buf(a.ws.blk_first, a.n_buf, g);
                const unsigned long long k = g - a.ws.blk_first[i], n = buf_count(a, i);
                m = (int)min((unsigned long long)kBlk, n - kBlk * k);
                xoff = buf_start(a, i) + kBlk * k;
            }
            s_m[j] = m; s_buf[j] = i; s_xoff[j] = xoff; s_key[j] = 0;
        }
        __syncthreads();

        // ---- pass A: sizes
        for (int j0 = warp * kQuadBlocks; j0 < kTileR; j0 += kWarps * kQuadBlocks) {
            if (s_m[j0] <= 0) break;                             // blocks of a tile are dense from 0
            const int j = j0 + q, m = s_m[j];
            T v[8][4], d[8][4];
            quad_load<W>(ids + s_xoff[j], m, true, v);
            quad_deltas<W>(v, m, d);
            uint32_t key;
            if constexpr (W == 32) {
                key = quad_choose_b<32, uint32_t>(d);
            } else {
                uint64_t o = 0;
#pragma unroll
                for (int i = 0; i < 8; i++) o |= d[i][0] | d[i][1] | d[i][2] | d[i][3];
                if (__all_sync(kFull, (o >> 32) == 0)) {
                    uint32_t d32[8][4];
#pragma unroll
                    for (int i = 0; i < 8; i++)
#pragma unroll
                        for (int c = 0; c < 4; c++) d32[i][c] = (uint32_t)d[i][c];
                    key = quad_choose_b<64, uint32_t>(d32);
                } else {
                    key = quad_choose_b<64, uint64_t>(d);
                }
            }
            if (l == 0) s_key[j] = m > 0 ? key : 0u;
        }
        __syncthreads();

        // ---- E3: intra-tile scan (warp 0), then CTA-wide decoupled look-back
        if (warp == 0) {
            uint32_t loc[kTileR / 32], sum = 0;
#pragma unroll
            for (int x = 0; x < kTileR / 32; x++) { loc[x] = sum; sum += s_key[lane * (kTileR / 32) + x] >> 18; }
            uint32_t inc = sum;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                uint32_t y = __shfl_up_sync(kFull, inc, o);
                if (lane >= o) inc += y;
            }
            const uint32_t base = inc - sum;
#pragma unroll
            for (int x = 0; x < kTileR / 32; x++) s_excl[lane * (kTileR / 32) + x] = base + loc[x];
            if (lane == 31) {
                s_excl[kTileR] = inc;
                if (t > 0) st_volatile_u64(&a.ws.tile_state[t], kFlagAgg | (unsigned long long)inc);
            }
        }
        unsigned long long excl = 0;
        if (t > 0) {
            long long idx = (long long)t - 1;
            while (true) {                                       // kThreads predecessors per round
                const long long mine = idx - tid;
                unsigned long long s = kFlagPre;                 // before tile 0: prefix 0
                if (mine >= 0) {
                    do { s = ld_volatile_u64(&a.ws.tile_state[mine]); } while ((s >> 62) == 0);
                }
                const uint32_t pre = __ballot_sync(kFull, (s >> 62) == 2);
                const int stop = __ffs(pre) - 1;
                unsigned long long val = (stop < 0 || lane <= stop) ? (s & kValMask) : 0ull;
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) val += __shfl_xor_sync(kFull, val, o);
                if (lane == 0) { s_lb_sum[warp] = val; s_lb_hit[warp] = stop >= 0; }
                __syncthreads();
                bool hit = false;
#pragma unroll
                for (int w2 = 0; w2 < kWarps; w2++) {
                    if (!hit) { excl += s_lb_sum[w2]; hit = s_lb_hit[w2] != 0; }
                }
                __syncthreads();
                if (hit) break;
                idx -= kThreads;
            }
        } else {
            __syncthreads();
        }
        if (tid == 0) {
            const unsigned long long agg = s_excl[kTileR];
            st_volatile_u64(&a.ws.tile_state[t], kFlagPre | (excl + agg));
            if (t == n_tiles - 1) {
                a.ws.hdr->grand16 = excl + agg;
                a.ws.hdr->total_out = a.ws.hdr->fixed_total + 16ull * (excl + agg);
            }
        }

        // ---- pass B: pack + emit
        for (int j0 = warp * kQuadBlocks; j0 < kTileR; j0 += kWarps * kQuadBlocks) {
            if (s_m[j0] <= 0) break;
            const int j = j0 + q, m = s_m[j];
            const uint32_t key = s_key[j];
            const uint32_t b = m > 0 ? 64u - ((key >> 7) & 127u) : 0u, n_exc = key & 127u;
            uint32_t* vq = st.vals + q * QuadStage<W>::kValWords;
            unsigned char* oq = st.out + q * QuadStage<W>::kOutStride;
            {
                T v[8][4], d[8][4];
                quad_load<W>(ids + s_xoff[j], m, false, v);
                quad_deltas<W>(v, m, d);
                if (l == 0) {                                    // block header (FORMAT.md §2)
                    reinterpret_cast<unsigned long long*>(oq)[0] = (unsigned long long)v[0][0];
                    reinterpret_cast<unsigned long long*>(oq)[1] = (unsigned long long)(b | (n_exc << 8));
                }
                if (__any_sync(kFull, n_exc > 0)) quad_exceptions<W, T>(vq, oq, d, b, n_exc);
                if constexpr (W == 32) {
                    quad_stage_vals<uint32_t>(vq, d, b);
                } else {
                    if (__any_sync(kFull, b > 32)) {             // wide payload somewhere in the batch
                        quad_stage_vals<uint64_t>(vq, d, b);
                        __syncwarp();
                        quad_pack_column64(reinterpret_cast<const uint64_t*>(vq) + l,
                                           reinterpret_cast<uint32_t*>(oq) + 4 + l, b);
                    } else {
                        uint32_t d32[8][4];
#pragma unroll
                        for (int i = 0; i < 8; i++)
#pragma unroll
                            for (int c = 0; c < 4; c++) d32[i][c] = (uint32_t)d[i][c];
                        quad_stage_vals<uint32_t>(vq, d32, b);
                        __syncwarp();
                        quad_pack_column32(vq + l, reinterpret_cast<uint32_t*>(oq) + 4 + l, b);
                    }
                }
            }
            if constexpr (W == 32) {
                __syncwarp();
                quad_pack_column32(vq + l, reinterpret_cast<uint32_t*>(oq) + 4 + l, b);
            }
            __syncwarp();

            // emit: final offsets, 128-bit stores, directory entry, stream start
            if (m > 0) {
                const uint32_t i = s_buf[j];
                const unsigned long long g = g0 + j;
                const unsigned long long first = a.ws.blk_first[i];
                const unsigned long long f0 = a.ws.fixed_prefix[i], f1 = a.ws.fixed_prefix[i + 1];
                const unsigned long long at = f1 + 16ull * (excl + s_excl[j]);
                const uint32_t bytes = key >> 14;
                unsigned long long S;
                if (first >= g0) S = f0 + 16ull * (excl + s_excl[first - g0]);
                else if (i == 0) S = 0;
                else {                                           // published by the tile that owns the first block
                    do { S = ld_volatile_u64(&a.ws.stream_start[i]); } while (S == 0);
                    S -= 1;
                }
                if (at + bytes <= a.out_cap) {
                    const uint4* src = reinterpret_cast<const uint4*>(oq);
                    uint4* dst = reinterpret_cast<uint4*>(a.out + at);
                    for (uint32_t x = l; x < bytes / 16; x += 4) __stcs(dst + x, src[x]);
                    if (l == 0) reinterpret_cast<uint32_t*>(a.out + S + 32)[g - first] = (uint32_t)((at - S) >> 4);
                } else if (l == 0) {
                    set_status(a.status, BFSC_ERR_DST_TOO_SMALL);
                }
                if (l == 0 && g == first) st_volatile_u64(&a.ws.stream_start[i], S + 1);
            }
            __syncwarp();
        }
    }
}

// ---- stream headers, directory tails, E5 raw passthrough, out_offsets --------------------
template <int W>
__global__ void __launch_bounds__(256) k_enc_streams(EncArgs a) {
    using T = typename IdT<W>::T;
    constexpr unsigned long long E = W / 8;
    const unsigned long long total_blocks = a.ws.hdr->total_blocks, grand16 = a.ws.hdr->grand16;
    bool ok = a.ws.hdr->ok != 0;
    if (ok && a.ws.hdr->total_out > a.out_cap) {
        ok = false;
        if (blockIdx.x == 0 && threadIdx.x == 0) set_status(a.status, BFSC_ERR_DST_TOO_SMALL);
    }
    // byte offset of stream i = fixed_prefix[i] + 16 * (scan value at its first block)
    auto stream_at = [&](uint32_t i) -> unsigned long long {
        const unsigned long long q = a.ws.blk_first[i];
        unsigned long long bb = grand16;
        if (q < total_blocks) {
            const uint32_t j = find_buf(a.ws.blk_first, a.n_buf, q);   // the buffer that owns block q
            bb = (a.ws.stream_start[j] - 1 - a.ws.fixed_prefix[j]) >> 4;
        }
        return a.ws.fixed_prefix[i] + 16ull * bb;
    };
    for (uint32_t i = blockIdx.x; i < a.n_buf; i += gridDim.x) {
        const unsigned long long f0 = a.ws.blk_first[i], f1 = a.ws.blk_first[i + 1];
        if (!ok) { if (a.out_off && threadIdx.x == 0) a.out_off[i] = 0; continue; }
        const unsigned long long s0 = stream_at(i);
        const unsigned long long s1 = (i + 1 < a.n_buf) ? stream_at(i + 1) : a.ws.hdr->total_out;
        const unsigned long long n = buf_count(a, i), total = s1 - s0;
        const bool raw = n * E < a.thr;
        unsigned char* s = a.out + s0;
        if (threadIdx.x == 0) {
            if (a.out_off) a.out_off[i] = s0;
            const unsigned long long nb = f1 - f0;
            uint4 h0, h1;
            h0.x = 0x43534642u;                                           // "BFSC"
            h0.y = 1u | ((uint32_t)W << 8) | ((raw ? 0u : 1u) << 16);
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
            for (unsigned long long j = threadIdx.x; j < padded; j += blockDim.x) y[j] = j < n ? x[j] : (T)0;
        }
    }
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        const unsigned long long t = ok ? a.ws.hdr->total_out : 0ull;
        if (a.out_off) a.out_off[a.n_buf] = t;
        if (a.out_total) *a.out_total = t;
    }
}

template <int W>
static bfsc_status launch_encode(const EncArgs& a, cudaStream_t s) {
    constexpr int kThreads = EncCfg<W>::kWarps * 32;
    constexpr size_t kSmem = sizeof(QuadStage<W>) * EncCfg<W>::kWarps;
    static int grid = 0;                          // persistent grid: all CTAs resident
    if (grid == 0) {
        int per_sm = 0, dev = 0, sms = kNumSM;
        if (cudaFuncSetAttribute(k_enc_fused<W>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmem) != cudaSuccess)
            return BFSC_ERR_CUDA;
        if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_enc_fused<W>, kThreads, kSmem) != cudaSuccess ||
            per_sm < 1)
            per_sm = 1;
        cudaGetDevice(&dev);
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        grid = sms * per_sm;
    }
    k_enc_plan<W><<<1, 1024, 0, s>>>(a);
    BFSC_LAUNCH_CHECK();
    k_enc_fused<W><<<grid, kThreads, kSmem, s>>>(a);
    BFSC_LAUNCH_CHECK();
    const uint32_t sgrid = a.n_buf < (uint32_t)(kNumSM * 8) ? a.n_buf : (uint32_t)(kNumSM * 8);
    k_enc_streams<W><<<sgrid ? sgrid : 1, 256, 0, s>>>(a);
    BFSC_LAUNCH_CHECK();
    return BFSC_OK;
}

static bfsc_status encode_common(const void* d_ids, const uint64_t* d_in_off, size_t n_single, size_t n_buf,
                                 bfsc_dtype t, size_t thr, void* d_out, size_t out_cap, uint64_t* d_out_off,
                                 uint64_t* d_out_total, void* ws, size_t ws_bytes, uint32_t* d_status, void* stream) {
    if (t != BFSC_U32 && t != BFSC_U64) return BFSC_ERR_INVALID_ARG;
    if (!d_out || !ws || n_buf > 0x7fffffffu) return BFSC_ERR_INVALID_ARG;
    if (((uintptr_t)d_ids & 15) || ((uintptr_t)d_out & 15) || ((uintptr_t)ws & 15)) return BFSC_ERR_INVALID_ARG;
    if (!d_ids && (d_in_off || n_single)) return BFSC_ERR_INVALID_ARG;
    EncArgs a;
    if (!ws_carve(ws, ws_bytes, n_buf, &a.ws)) return BFSC_ERR_INVALID_ARG;
    a.ids = d_ids; a.in_off = (const unsigned long long*)d_in_off; a.n_single = n_single;
    a.n_buf = (uint32_t)n_buf; a.thr = thr; a.out = (unsigned char*)d_out; a.out_cap = out_cap;
    a.out_off = (unsigned long long*)d_out_off; a.out_total = (unsigned long long*)d_out_total; a.status = d_status;
    return t == BFSC_U32 ? launch_encode<32>(a, (cudaStream_t)stream) : launch_encode<64>(a, (cudaStream_t)stream);
}

}  // namespace bfsc

extern "C" bfsc_status bfsc_compress(const void* d_ids, size_t n_ids, bfsc_dtype t, size_t raw_threshold_bytes,
                                     void* d_out, size_t out_capacity, uint64_t* d_out_bytes, void* d_workspace,
                                     size_t workspace_bytes, uint32_t* d_status, void* cuda_stream) {
    if (!d_out_bytes) return BFSC_ERR_INVALID_ARG;
    return bfsc::encode_common(d_ids, nullptr, n_ids, 1, t, raw_threshold_bytes, d_out, out_capacity, nullptr,
                               d_out_bytes, d_workspace, workspace_bytes, d_status, cuda_stream);
}

extern "C" bfsc_status bfsc_compress_batch(const void* d_ids, const uint64_t* d_in_offsets, size_t n_buf,
                                           bfsc_dtype t, size_t raw_threshold_bytes, void* d_out,
                                           size_t out_capacity, uint64_t* d_out_offsets, void* d_workspace,
                                           size_t workspace_bytes, uint32_t* d_status, void* cuda_stream) {
    if (!d_in_offsets || !d_out_offsets) return BFSC_ERR_INVALID_ARG;
    return bfsc::encode_common(d_ids, d_in_offsets, 0, n_buf, t, raw_threshold_bytes, d_out, out_capacity,
                               d_out_offsets, nullptr, d_workspace, workspace_bytes, d_status, cuda_stream);
}
