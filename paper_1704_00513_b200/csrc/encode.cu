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
    if (threadIdx.x == 0) {
        a.ws.blk_first[a.n_buf] = carry.a;
        a.ws.fixed_prefix[a.n_buf] = carry.b;
        a.ws.stream_start[a.n_buf] = 0;
        a.ws.hdr->total_blocks = carry.a;
        a.ws.hdr->fixed_total = carry.b;
        a.ws.hdr->ticket = 0;
        const bool ok = !bad && carry.a <= a.ws.blk_cap;
        a.ws.hdr->ok = ok ? 1u : 0u;
        if (!ok) set_status(a.status, BFSC_ERR_INVALID_ARG);
    }
}

// ---- E1+E2 per block: sizes ------------------------------------------------------------
template <int W>
__global__ void __launch_bounds__(256) k_enc_analyze(EncArgs a) {
    using T = typename IdT<W>::T;
    if (!a.ws.hdr->ok) return;
    const unsigned long long total = a.ws.hdr->total_blocks;
    const unsigned long long nwarps = (unsigned long long)gridDim.x * (blockDim.x >> 5);
    for (unsigned long long g = (unsigned long long)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5); g < total;
         g += nwarps) {
        const uint32_t i = find_buf(a.ws.blk_first, a.n_buf, g);
        const unsigned long long k = g - a.ws.blk_first[i], n = buf_count(a, i);
        const int m = (int)min((unsigned long long)kBlk, n - kBlk * k);
        const T* x = reinterpret_cast<const T*>(a.ids) + buf_start(a, i) + kBlk * k;
        T v[4], d[4];
        int w[4];
        load_rows<W>(x, m, v);
        deltas<W>(v, m, d);
        widths_of<W>(d, w);
        const uint32_t key = choose_b<W>(w);
        if (lane_id() == 0) {
            const uint32_t cost = key >> 14, b = 64u - ((key >> 7) & 127u), n_exc = key & 127u;
            a.ws.meta[g] = (cost >> 4) | (b << 8) | (n_exc << 16);
        }
    }
}

// ---- E3: exclusive scan of the block sizes (16-byte units), one CTA ----------------------
__global__ void __launch_bounds__(1024) k_enc_scan(EncArgs a) {
    __shared__ Scan2 sm[33];
    if (!a.ws.hdr->ok) return;
    const unsigned long long total = a.ws.hdr->total_blocks;
    unsigned long long carry = 0;
    for (unsigned long long g0 = 0; g0 < total; g0 += blockDim.x) {
        const unsigned long long g = g0 + threadIdx.x;
        Scan2 v{g < total ? (unsigned long long)(a.ws.meta[g] & 0xffu) : 0ull, 0ull};
        Scan2 tot;
        Scan2 ex = block_scan_excl2(v, &tot, sm);
        if (g < total) a.ws.bb16[g] = (uint32_t)(carry + ex.a);
        carry += tot.a;
    }
    if (threadIdx.x == 0) {
        a.ws.bb16[total] = (uint32_t)carry;
        const unsigned long long out_total = a.ws.hdr->fixed_total + 16ull * carry;
        a.ws.hdr->total_out = out_total;
        if (out_total > a.out_cap || carry > 0xffffffffull) {
            a.ws.hdr->ok = 0;
            set_status(a.status, BFSC_ERR_DST_TOO_SMALL);
        }
    }
}

// ---- E4: pack + emit blocks and directory entries ---------------------------------------
template <int W>
__global__ void __launch_bounds__(256) k_enc_pack(EncArgs a) {
    using T = typename IdT<W>::T;
    __shared__ EncStage<W> stage[8];
    if (!a.ws.hdr->ok) return;
    EncStage<W>& st = stage[threadIdx.x >> 5];
    const unsigned long long total = a.ws.hdr->total_blocks;
    const unsigned long long nwarps = (unsigned long long)gridDim.x * (blockDim.x >> 5);
    for (unsigned long long g = (unsigned long long)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5); g < total;
         g += nwarps) {
        const uint32_t i = find_buf(a.ws.blk_first, a.n_buf, g);
        const unsigned long long first = a.ws.blk_first[i];
        const unsigned long long k = g - first, n = buf_count(a, i);
        const int m = (int)min((unsigned long long)kBlk, n - kBlk * k);
        const T* x = reinterpret_cast<const T*>(a.ids) + buf_start(a, i) + kBlk * k;
        T v[4], d[4];
        load_rows<W>(x, m, v);
        const T base = deltas<W>(v, m, d);
        const uint32_t meta = a.ws.meta[g];
        const uint32_t b = (meta >> 8) & 0xffu, n_exc = (meta >> 16) & 0xffu;
        const uint32_t bytes = pack_block<W>(st, d, base, b, n_exc);
        const unsigned long long stream = a.ws.fixed_prefix[i] + 16ull * a.ws.bb16[first];
        const unsigned long long at = a.ws.fixed_prefix[i + 1] + 16ull * a.ws.bb16[g];
        store_block<W>(st, a.out + at, bytes);
        if (lane_id() == 0)
            reinterpret_cast<uint32_t*>(a.out + stream + 32)[k] = (uint32_t)((at - stream) >> 4);
        __syncwarp();
    }
}

// ---- stream headers, directory tails, E5 raw passthrough, out_offsets --------------------
template <int W>
__global__ void __launch_bounds__(256) k_enc_streams(EncArgs a) {
    using T = typename IdT<W>::T;
    constexpr unsigned long long E = W / 8;
    const bool ok = a.ws.hdr->ok != 0;
    for (uint32_t i = blockIdx.x; i < a.n_buf; i += gridDim.x) {
        const unsigned long long f0 = a.ws.blk_first[i], f1 = a.ws.blk_first[i + 1];
        if (!ok) { if (a.out_off && threadIdx.x == 0) a.out_off[i] = 0; continue; }
        const unsigned long long s0 = a.ws.fixed_prefix[i] + 16ull * a.ws.bb16[f0];
        const unsigned long long s1 = a.ws.fixed_prefix[i + 1] + 16ull * a.ws.bb16[f1];
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
    const int grid = kNumSM * 8;
    k_enc_plan<W><<<1, 1024, 0, s>>>(a);
    BFSC_LAUNCH_CHECK();
    k_enc_analyze<W><<<grid, 256, 0, s>>>(a);
    BFSC_LAUNCH_CHECK();
    k_enc_scan<<<1, 1024, 0, s>>>(a);
    BFSC_LAUNCH_CHECK();
    k_enc_pack<W><<<grid, 256, 0, s>>>(a);
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
