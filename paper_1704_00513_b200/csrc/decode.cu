// decode.cu — bfsc_decompress / bfsc_decompress_batch (steps D0-D5).
#include "block_decode.cuh"

namespace bfsc {

struct DecArgs {
    const unsigned char* in;
    const unsigned long long* in_off;   // n_buf+1 byte offsets, or nullptr (single stream, in_single bytes)
    unsigned long long in_single;
    uint32_t n_buf;
    void* ids;
    unsigned long long ids_cap;
    unsigned long long* id_off;         // n_buf+1 (batch, written) or nullptr
    unsigned long long* n_ids_out;      // single: *d_n_ids, or nullptr
    uint32_t* status;
    WsView ws;                          // blk_first, fixed_prefix (= id offsets)
};

__device__ __forceinline__ unsigned long long s_begin(const DecArgs& a, uint32_t i) {
    return a.in_off ? a.in_off[i] : 0ull;
}
__device__ __forceinline__ unsigned long long s_avail(const DecArgs& a, uint32_t i) {
    return a.in_off ? a.in_off[i + 1] - a.in_off[i] : a.in_single;
}

// ---- D0: plan. Parse + validate every stream header; prefixes of IDs and blocks. ----------
template <int W>
__global__ void __launch_bounds__(1024) k_dec_plan(DecArgs a) {
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
            const unsigned long long beg = s_begin(a, i);
            unsigned long long avail = 0;
            bool ok = true;
            if (a.in_off && a.in_off[i + 1] < beg) ok = false; else avail = s_avail(a, i);
            if ((beg & 15) || avail < 32) ok = false;
            if (ok) {
                const uint4 h0 = *reinterpret_cast<const uint4*>(a.in + beg);
                const uint4 h1 = *reinterpret_cast<const uint4*>(a.in + beg + 16);
                const uint32_t mode = (h0.y >> 16) & 0xffu;
                const unsigned long long n = (unsigned long long)h0.w << 32 | h0.z;
                const unsigned long long total = (unsigned long long)h1.y << 32 | h1.x;
                const unsigned long long nb = h1.z;
                if (h0.x != 0x43534642u || (h0.y & 0xffu) != 1u || ((h0.y >> 8) & 0xffu) != (uint32_t)W ||
                    mode > 1u || (h0.y >> 24) != 0u)
                    ok = false;
                else if (total > avail || (total & 15) || total < 32) ok = false;
                else if (mode == 0) { if (nb != 0 || n > (total - 32) / E) ok = false; }
                else if (nb != (n + kBlk - 1) / kBlk || n > (1ull << 40) ||
                         32ull + ((4ull * (nb + 1) + 15ull) & ~15ull) > total)
                    ok = false;
                if (ok) { v.a = nb; v.b = n; }
            }
            if (!ok) bad = 1;
        }
        Scan2 tot;
        Scan2 ex = block_scan_excl2(v, &tot, sm);
        if (i < a.n_buf) {
            a.ws.blk_first[i] = carry.a + ex.a;
            a.ws.fixed_prefix[i] = carry.b + ex.b;
        }
        carry.a += tot.a; carry.b += tot.b;
    }
    __syncthreads();
    const bool good = !bad && carry.a <= a.ws.blk_cap && carry.b <= a.ids_cap;
    if (threadIdx.x == 0) {
        a.ws.blk_first[a.n_buf] = carry.a;
        a.ws.fixed_prefix[a.n_buf] = carry.b;
        a.ws.hdr->total_blocks = carry.a;
        a.ws.hdr->total_out = carry.b;
        a.ws.hdr->ok = good ? 1u : 0u;
        if (bad) set_status(a.status, BFSC_ERR_CORRUPT);
        else if (carry.b > a.ids_cap) set_status(a.status, BFSC_ERR_DST_TOO_SMALL);
        else if (!good) set_status(a.status, BFSC_ERR_INVALID_ARG);
        if (a.n_ids_out) *a.n_ids_out = good ? carry.b : 0ull;
    }
    __syncthreads();
    if (a.id_off)
        for (uint32_t i = threadIdx.x; i <= a.n_buf; i += blockDim.x) a.id_off[i] = good ? a.ws.fixed_prefix[i] : 0ull;
}

// ---- D1-D4 per block -------------------------------------------------------------------
template <int W>
__global__ void __launch_bounds__(256) k_dec_blocks(DecArgs a) {
    using T = typename IdT<W>::T;
    if (!a.ws.hdr->ok) return;
    const unsigned long long total_blocks = a.ws.hdr->total_blocks;
    const unsigned long long nwarps = (unsigned long long)gridDim.x * (blockDim.x >> 5);
    for (unsigned long long g = (unsigned long long)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
         g < total_blocks; g += nwarps) {
        const uint32_t i = find_buf(a.ws.blk_first, a.n_buf, g);
        const unsigned long long k = g - a.ws.blk_first[i];
        const unsigned long long id0 = a.ws.fixed_prefix[i], n = a.ws.fixed_prefix[i + 1] - id0;
        const unsigned char* s = a.in + s_begin(a, i);
        const unsigned long long total16 = *reinterpret_cast<const unsigned long long*>(s + 16) >> 4;
        const unsigned long long nb = (n + kBlk - 1) / kBlk;
        const uint32_t* dir = reinterpret_cast<const uint32_t*>(s + 32);
        const unsigned long long o0 = dir[k], o1 = dir[k + 1];
        const unsigned long long lo16 = (32ull + ((4ull * (nb + 1) + 15ull) & ~15ull)) >> 4;
        if (o0 < lo16 || o1 <= o0 || o1 > total16) { set_status(a.status, BFSC_ERR_CORRUPT); continue; }
        const unsigned char* blk = s + 16ull * o0;
        const uint4 h = *reinterpret_cast<const uint4*>(blk);
        const uint32_t b = h.z & 0xffu, n_exc = (h.z >> 8) & 0xffu;
        if (b > (uint32_t)W || n_exc > 127u || 16ull + 16ull * b + exc_bytes<W>(n_exc) > 16ull * (o1 - o0)) {
            set_status(a.status, BFSC_ERR_CORRUPT);
            continue;
        }
        const T base = (T)((unsigned long long)h.y << 32 | h.x);
        T d[4];
        unpack_rows<W>(reinterpret_cast<const uint4*>(blk + 16), b, d);
        if (n_exc > 0 && !patch_rows<W>(blk + 16 + 16 * b, b, n_exc, d)) {
            set_status(a.status, BFSC_ERR_CORRUPT);
            continue;
        }
        const int m = (int)min((unsigned long long)kBlk, n - kBlk * k);
        scan_store<W>(d, base, reinterpret_cast<T*>(a.ids) + id0 + kBlk * k, m);
    }
}

// ---- D5 raw passthrough -----------------------------------------------------------------
template <int W>
__global__ void __launch_bounds__(256) k_dec_raw(DecArgs a) {
    using T = typename IdT<W>::T;
    if (!a.ws.hdr->ok) return;
    for (uint32_t i = blockIdx.x; i < a.n_buf; i += gridDim.x) {
        const unsigned char* s = a.in + s_begin(a, i);
        if (s[6] != 0) continue;
        const unsigned long long id0 = a.ws.fixed_prefix[i], n = a.ws.fixed_prefix[i + 1] - id0;
        const T* x = reinterpret_cast<const T*>(s + 32);
        T* y = reinterpret_cast<T*>(a.ids) + id0;
        for (unsigned long long j = threadIdx.x; j < n; j += blockDim.x) y[j] = x[j];
    }
}

template <int W>
static bfsc_status launch_decode(const DecArgs& a, cudaStream_t s) {
    const int grid = kNumSM * 8;
    k_dec_plan<W><<<1, 1024, 0, s>>>(a);
    BFSC_LAUNCH_CHECK();
    k_dec_blocks<W><<<grid, 256, 0, s>>>(a);
    BFSC_LAUNCH_CHECK();
    const uint32_t rgrid = a.n_buf < (uint32_t)(kNumSM * 8) ? a.n_buf : (uint32_t)(kNumSM * 8);
    k_dec_raw<W><<<rgrid ? rgrid : 1, 256, 0, s>>>(a);
    BFSC_LAUNCH_CHECK();
    return BFSC_OK;
}

static bfsc_status decode_common(const void* d_in, const uint64_t* d_in_off, size_t in_single, size_t n_buf,
                                 bfsc_dtype t, void* d_ids, size_t ids_cap, uint64_t* d_id_off, uint64_t* d_n_ids,
                                 void* ws, size_t ws_bytes, uint32_t* d_status, void* stream) {
    if (t != BFSC_U32 && t != BFSC_U64) return BFSC_ERR_INVALID_ARG;
    if (!d_in || !ws || n_buf > 0x7fffffffu) return BFSC_ERR_INVALID_ARG;
    if (!d_ids && ids_cap) return BFSC_ERR_INVALID_ARG;
    if (((uintptr_t)d_in & 15) || ((uintptr_t)d_ids & 15) || ((uintptr_t)ws & 15)) return BFSC_ERR_INVALID_ARG;
    DecArgs a;
    if (!ws_carve(ws, ws_bytes, n_buf, &a.ws)) return BFSC_ERR_INVALID_ARG;
    a.in = (const unsigned char*)d_in; a.in_off = (const unsigned long long*)d_in_off; a.in_single = in_single;
    a.n_buf = (uint32_t)n_buf; a.ids = d_ids; a.ids_cap = ids_cap; a.id_off = (unsigned long long*)d_id_off;
    a.n_ids_out = (unsigned long long*)d_n_ids; a.status = d_status;
    return t == BFSC_U32 ? launch_decode<32>(a, (cudaStream_t)stream) : launch_decode<64>(a, (cudaStream_t)stream);
}

}  // namespace bfsc

extern "C" bfsc_status bfsc_decompress(const void* d_in, size_t in_bytes, bfsc_dtype t, void* d_ids,
                                       size_t ids_capacity, uint64_t* d_n_ids, void* d_workspace,
                                       size_t workspace_bytes, uint32_t* d_status, void* cuda_stream) {
    if (!d_n_ids) return BFSC_ERR_INVALID_ARG;
    return bfsc::decode_common(d_in, nullptr, in_bytes, 1, t, d_ids, ids_capacity, nullptr, d_n_ids, d_workspace,
                               workspace_bytes, d_status, cuda_stream);
}

extern "C" bfsc_status bfsc_decompress_batch(const void* d_in, const uint64_t* d_in_offsets, size_t n_buf,
                                             bfsc_dtype t, void* d_ids, size_t ids_capacity,
                                             uint64_t* d_id_offsets, void* d_workspace, size_t workspace_bytes,
                                             uint32_t* d_status, void* cuda_stream) {
    if (!d_in_offsets || !d_id_offsets) return BFSC_ERR_INVALID_ARG;
    return bfsc::decode_common(d_in, d_in_offsets, 0, n_buf, t, d_ids, ids_capacity, d_id_offsets, nullptr,
                               d_workspace, workspace_bytes, d_status, cuda_stream);
}
