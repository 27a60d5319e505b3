// encode.cu — bfsc_compress / bfsc_compress_batch (steps E0-E5).
#include "block_encode.cuh"

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
    constexpr unsigned long long kTile = (W == 32) ? 32 : 16;   // = 8 * FusedCfg<W>::kBpw
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

// ---- E1-E4 fused: one pass over the input ------------------------------------------------
// Persistent CTAs pull tiles of kBpw*8 consecutive blocks by ticket. 8 worker warps each own
// kBpw blocks (warp = block); a 9th warp owns the bookkeeping: block -> buffer mapping, the
// intra-tile scan of block sizes and the decoupled look-back that turns it into the device-wide
// exclusive scan (E3) while the workers already pack into shared memory.
template <int W> struct FusedCfg { static constexpr int kBpw = (W == 32) ? 4 : 2; };

struct BlkMeta {
    unsigned long long xoff;     // element offset of the block's first ID in ids
    unsigned long long first;    // first global block of its buffer
    unsigned long long f0, f1;   // fixed_prefix[i], fixed_prefix[i+1]
    uint32_t i;                  // buffer
    int m;                       // valid IDs (0 = no such block)
};

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
__global__ void __launch_bounds__(288) k_enc_fused(EncArgs a) {
    using T = typename IdT<W>::T;
    constexpr int kBpw = FusedCfg<W>::kBpw, kTile = 8 * kBpw;
    struct Stage {
        alignas(16) T vals[kBlk];
        alignas(16) unsigned char out[kBpw][EncStage<W>::kOutBytes];
    };
    __shared__ Stage stage[8];
    __shared__ BlkMeta meta[2][kTile];
    __shared__ uint32_t sm_size16[kTile];
    __shared__ uint32_t sm_excl[kTile + 1];
    __shared__ unsigned long long sm_tile_excl;
    __shared__ unsigned long long sm_tile[2];

    if (!a.ws.hdr->ok) return;
    const unsigned long long total = a.ws.hdr->total_blocks;
    const unsigned long long n_tiles = (total + kTile - 1) / kTile;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const bool is_scan = (warp == 8);

    for (int it = 0;; it++) {
        const int par = it & 1;
        if (is_scan) {                                   // ticket + block metadata of the tile
            unsigned long long t = 0;
            if (lane == 0) t = atomicAdd(&a.ws.hdr->ticket, 1u);
            t = __shfl_sync(kFull, t, 0);
            if (lane == 0) sm_tile[par] = t;
            const unsigned long long g = t * kTile + lane;
            if (lane < kTile) {
                BlkMeta mt;
                mt.m = 0; mt.i = 0; mt.xoff = 0; mt.first = 0; mt.f0 = 0; mt.f1 = 0;
                if (t < n_tiles && g < total) {
                    const uint32_t i = find_buf(a.ws.blk_first, a.n_buf, g);
                    mt.i = i;
                    mt.first = a.ws.blk_first[i];
                    const unsigned long long k = g - mt.first, n = buf_count(a, i);
                    mt.m = (int)min((unsigned long long)kBlk, n - kBlk * k);
                    mt.xoff = buf_start(a, i) + kBlk * k;
                    mt.f0 = a.ws.fixed_prefix[i];
                    mt.f1 = a.ws.fixed_prefix[i + 1];
                }
                meta[par][lane] = mt;
            }
        }
        __syncthreads();                                 // S1
        const unsigned long long t = sm_tile[par];
        if (t >= n_tiles) break;
        const unsigned long long g0 = t * kTile;

        T d[kBpw][4];
        T base[kBpw];
        uint32_t key[kBpw];
        if (!is_scan) {                                  // E1 + E2
            T v[kBpw][4];
#pragma unroll
            for (int q = 0; q < kBpw; q++) {
                const BlkMeta& mt = meta[par][warp * kBpw + q];
                if (mt.m > 0) load_rows<W>(reinterpret_cast<const T*>(a.ids) + mt.xoff, mt.m, v[q]);
                else v[q][0] = v[q][1] = v[q][2] = v[q][3] = 0;
            }
#pragma unroll
            for (int q = 0; q < kBpw; q++) {
                const int m = meta[par][warp * kBpw + q].m;
                base[q] = deltas<W>(v[q], m > 0 ? m : 1, d[q]);
                int w[4];
                widths_of<W>(d[q], w);
                key[q] = choose_b<W>(w);
                if (lane == 0) sm_size16[warp * kBpw + q] = m > 0 ? (key[q] >> 18) : 0u;   // (cost >> 4)
            }
        }
        __syncthreads();                                 // S2
        if (is_scan) {                                   // E3: intra-tile scan, then look-back
            uint32_t sz = lane < kTile ? sm_size16[lane] : 0u, inc = sz;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                uint32_t x = __shfl_up_sync(kFull, inc, o);
                if (lane >= o) inc += x;
            }
            if (lane < kTile) sm_excl[lane] = inc - sz;
            const unsigned long long agg = __shfl_sync(kFull, inc, 31);
            if (lane == 0) {
                sm_excl[kTile] = (uint32_t)agg;
                if (t > 0) st_volatile_u64(&a.ws.tile_state[t], kFlagAgg | agg);
            }
            unsigned long long excl = 0;
            if (t > 0) {
                long long idx = (long long)t - 1;
                while (true) {
                    const long long mine = idx - lane;
                    unsigned long long s = kFlagPre;     // tiles before 0: prefix 0
                    if (mine >= 0) {
                        do { s = ld_volatile_u64(&a.ws.tile_state[mine]); } while ((s >> 62) == 0);
                    }
                    const uint32_t pre = __ballot_sync(kFull, (s >> 62) == 2);
                    const int stop = __ffs(pre) - 1;     // nearest tile with a full prefix (always exists: idx<0 lanes)
                    unsigned long long val = (stop < 0 || lane <= stop) ? (s & kValMask) : 0ull;
#pragma unroll
                    for (int o = 16; o > 0; o >>= 1) val += __shfl_xor_sync(kFull, val, o);
                    excl += val;
                    if (stop >= 0) break;
                    idx -= 32;
                }
            }
            if (lane == 0) {
                st_volatile_u64(&a.ws.tile_state[t], kFlagPre | (excl + agg));
                sm_tile_excl = excl;
                if (t == n_tiles - 1) {
                    a.ws.hdr->grand16 = excl + agg;
                    a.ws.hdr->total_out = a.ws.hdr->fixed_total + 16ull * (excl + agg);
                }
            }
        } else {                                         // E4: pack into shared memory meanwhile
#pragma unroll
            for (int q = 0; q < kBpw; q++) {
                if (meta[par][warp * kBpw + q].m > 0) {
                    const uint32_t b = 64u - ((key[q] >> 7) & 127u), n_exc = key[q] & 127u;
                    pack_block_to<W>(stage[warp].vals, stage[warp].out[q], d[q], base[q], b, n_exc);
                }
            }
        }
        __syncthreads();                                 // S3
        if (!is_scan) {                                  // emit: 128-bit coalesced stores + directory entries
            const unsigned long long tile_excl = sm_tile_excl;
#pragma unroll
            for (int q = 0; q < kBpw; q++) {
                const int blk = warp * kBpw + q;
                const BlkMeta& mt = meta[par][blk];
                if (mt.m <= 0) continue;
                const unsigned long long g = g0 + blk;
                const unsigned long long at = mt.f1 + 16ull * (tile_excl + sm_excl[blk]);
                const uint32_t bytes = (key[q] >> 14);
                unsigned long long S;
                if (mt.first >= g0) {
                    S = mt.f0 + 16ull * (tile_excl + sm_excl[mt.first - g0]);
                } else {
                    unsigned long long s1 = 0;
                    if (lane == 0) { do { s1 = ld_volatile_u64(&a.ws.stream_start[mt.i]); } while (s1 == 0); }
                    S = __shfl_sync(kFull, s1, 0) - 1;
                }
                if (at + bytes <= a.out_cap) {
                    const uint4* src = reinterpret_cast<const uint4*>(stage[warp].out[q]);
                    uint4* dst = reinterpret_cast<uint4*>(a.out + at);
                    for (uint32_t x = lane; x < bytes / 16; x += 32) __stcs(dst + x, src[x]);
                    if (lane == 0) reinterpret_cast<uint32_t*>(a.out + S + 32)[g - mt.first] = (uint32_t)((at - S) >> 4);
                } else if (lane == 0) {
                    set_status(a.status, BFSC_ERR_DST_TOO_SMALL);
                }
                if (lane == 0 && g == mt.first) st_volatile_u64(&a.ws.stream_start[mt.i], S + 1);
            }
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
    static int per_sm = 0;                        // persistent grid: every CTA resident (look-back needs it)
    if (per_sm == 0) {
        if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_enc_fused<W>, 288, 0) != cudaSuccess || per_sm < 1)
            per_sm = 1;
    }
    int dev = 0, sms = kNumSM;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    const int grid = sms * per_sm;
    k_enc_plan<W><<<1, 1024, 0, s>>>(a);
    BFSC_LAUNCH_CHECK();
    k_enc_fused<W><<<grid, 288, 0, s>>>(a);
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
