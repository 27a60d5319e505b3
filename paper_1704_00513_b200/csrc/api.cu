// api.cu — host-only entry points of the C ABI: bounds, workspace size, host-buffer calls.
#include "common.cuh"

#include <mutex>

namespace bfsc {
unsigned long long g_launches = 0;

bool current_device(DeviceInfo* d) {
    static std::mutex mu;
    static int sms[kMaxDevices] = {};
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kMaxDevices) return false;
    std::lock_guard<std::mutex> lock(mu);
    if (sms[dev] == 0) {
        int n = 0;
        if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n < 1) return false;
        sms[dev] = n;
    }
    d->device = dev;
    d->sms = sms[dev];
    return true;
}

static size_t bound_one(size_t n, int W) {
    const size_t nb = (n + kBlk - 1) / kBlk;
    const size_t pfor = 32 + align_up(4 * (nb + 1), 16) + nb * (16 + 16 * (size_t)W);
    const size_t raw = 32 + align_up(n * (size_t)(W / 8), 16);
    return pfor > raw ? pfor : raw;
}
}  // namespace bfsc

extern "C" uint32_t bfsc_version(void) { return (1u << 16) | 3u; }   // abi revision 2: bfsc_compress[_batch]_codec, mode 2; 3: codec flags, bitmap calls

extern "C" uint64_t bfsc_kernel_launches(void) { return bfsc::g_launches; }

extern "C" size_t bfsc_compress_bound(size_t n_ids, bfsc_dtype t) {
    if (t != BFSC_U32 && t != BFSC_U64) return 0;
    return bfsc::bound_one(n_ids, (int)t);
}

extern "C" size_t bfsc_batch_compress_bound(const uint64_t* h_counts, size_t n_buf, bfsc_dtype t) {
    if ((t != BFSC_U32 && t != BFSC_U64) || (!h_counts && n_buf)) return 0;
    size_t s = 0;
    for (size_t i = 0; i < n_buf; i++) s += bfsc::bound_one((size_t)h_counts[i], (int)t);
    return s;
}

extern "C" size_t bfsc_workspace_bytes(size_t n_ids_total, size_t n_buf, bfsc_dtype t) {
    (void)t;
    return bfsc::align_up(bfsc::ws_bytes_for(n_ids_total, n_buf), 256);
}

// standard workspace of one stream of at most n_bits IDs | the bitmap's rank tables (common.cuh)
extern "C" size_t bfsc_bitmap_workspace_bytes(size_t n_bits, bfsc_dtype t) {
    (void)t;
    return bfsc::align_up(bfsc::align_up(bfsc::ws_bytes_for(n_bits, 1), 16) + bfsc::bitmap_extra_ws_bytes(n_bits), 256);
}

// ---- host-buffer convenience calls ------------------------------------------------------
// scratch = [ids: align256(n*W/8)] [stream: align256(bound)] [workspace] [result: 256 B]
namespace bfsc {
struct HostLayout { size_t ids, stream, ws, res, total, ids_bytes, stream_bytes, ws_bytes; };
static HostLayout host_layout(size_t n, int W) {
    HostLayout L;
    L.ids_bytes = align_up(n * (size_t)(W / 8) + 16, 256);
    L.stream_bytes = align_up(bound_one(n, W), 256);
    L.ws_bytes = align_up(ws_bytes_for(n, 1), 256);
    L.ids = 0; L.stream = L.ids_bytes; L.ws = L.stream + L.stream_bytes; L.res = L.ws + L.ws_bytes;
    L.total = L.res + 256;
    return L;
}
}  // namespace bfsc

extern "C" size_t bfsc_host_scratch_bytes(size_t n_ids, bfsc_dtype t) {
    if (t != BFSC_U32 && t != BFSC_U64) return 0;
    return bfsc::host_layout(n_ids, (int)t).total;
}

extern "C" bfsc_status bfsc_compress_host(const void* h_ids, size_t n_ids, bfsc_dtype t, size_t raw_threshold_bytes,
                                          void* h_out, size_t out_capacity, uint64_t* h_out_bytes, void* d_scratch,
                                          size_t scratch_bytes, void* cuda_stream) {
    if (t != BFSC_U32 && t != BFSC_U64) return BFSC_ERR_INVALID_ARG;
    if (!h_out || !h_out_bytes || !d_scratch || (!h_ids && n_ids)) return BFSC_ERR_INVALID_ARG;
    const bfsc::HostLayout L = bfsc::host_layout(n_ids, (int)t);
    if (scratch_bytes < L.total || ((uintptr_t)d_scratch & 255)) return BFSC_ERR_INVALID_ARG;
    cudaStream_t s = (cudaStream_t)cuda_stream;
    char* base = (char*)d_scratch;
    uint64_t* d_res = (uint64_t*)(base + L.res);               // [0] = out bytes, [1] = status word
    if (cudaMemsetAsync(d_res, 0, 16, s) != cudaSuccess) return BFSC_ERR_CUDA;
    if (n_ids && cudaMemcpyAsync(base + L.ids, h_ids, n_ids * (size_t)(t / 8), cudaMemcpyHostToDevice, s) != cudaSuccess)
        return BFSC_ERR_CUDA;
    bfsc_status rc = bfsc_compress(base + L.ids, n_ids, t, raw_threshold_bytes, base + L.stream, L.stream_bytes,
                                   d_res, base + L.ws, L.ws_bytes, (uint32_t*)(d_res + 1), s);
    if (rc != BFSC_OK) return rc;
    uint64_t res[2];
    if (cudaMemcpyAsync(res, d_res, 16, cudaMemcpyDeviceToHost, s) != cudaSuccess) return BFSC_ERR_CUDA;
    if (cudaStreamSynchronize(s) != cudaSuccess) return BFSC_ERR_CUDA;
    if ((uint32_t)res[1]) return (bfsc_status)(uint32_t)res[1];
    if (res[0] > out_capacity) return BFSC_ERR_DST_TOO_SMALL;
    if (cudaMemcpyAsync(h_out, base + L.stream, res[0], cudaMemcpyDeviceToHost, s) != cudaSuccess) return BFSC_ERR_CUDA;
    if (cudaStreamSynchronize(s) != cudaSuccess) return BFSC_ERR_CUDA;
    *h_out_bytes = res[0];
    return BFSC_OK;
}

extern "C" bfsc_status bfsc_decompress_host(const void* h_in, size_t in_bytes, bfsc_dtype t, void* h_ids,
                                            size_t ids_capacity, uint64_t* h_n_ids, void* d_scratch,
                                            size_t scratch_bytes, void* cuda_stream) {
    if (t != BFSC_U32 && t != BFSC_U64) return BFSC_ERR_INVALID_ARG;
    if (!h_in || !h_n_ids || !d_scratch || in_bytes < 32 || (!h_ids && ids_capacity)) return BFSC_ERR_INVALID_ARG;
    const bfsc::HostLayout L = bfsc::host_layout(ids_capacity, (int)t);
    if (scratch_bytes < L.total || ((uintptr_t)d_scratch & 255)) return BFSC_ERR_INVALID_ARG;
    if (in_bytes > L.stream_bytes) in_bytes = L.stream_bytes;   // a stream of <= ids_capacity IDs cannot be larger
    cudaStream_t s = (cudaStream_t)cuda_stream;
    char* base = (char*)d_scratch;
    uint64_t* d_res = (uint64_t*)(base + L.res);
    if (cudaMemsetAsync(d_res, 0, 16, s) != cudaSuccess) return BFSC_ERR_CUDA;
    if (cudaMemcpyAsync(base + L.stream, h_in, in_bytes, cudaMemcpyHostToDevice, s) != cudaSuccess) return BFSC_ERR_CUDA;
    bfsc_status rc = bfsc_decompress(base + L.stream, in_bytes, t, base + L.ids, ids_capacity, d_res, base + L.ws,
                                     L.ws_bytes, (uint32_t*)(d_res + 1), s);
    if (rc != BFSC_OK) return rc;
    uint64_t res[2];
    if (cudaMemcpyAsync(res, d_res, 16, cudaMemcpyDeviceToHost, s) != cudaSuccess) return BFSC_ERR_CUDA;
    if (cudaStreamSynchronize(s) != cudaSuccess) return BFSC_ERR_CUDA;
    if ((uint32_t)res[1]) return (bfsc_status)(uint32_t)res[1];
    if (res[0] && cudaMemcpyAsync(h_ids, base + L.ids, res[0] * (size_t)(t / 8), cudaMemcpyDeviceToHost, s) != cudaSuccess)
        return BFSC_ERR_CUDA;
    if (cudaStreamSynchronize(s) != cudaSuccess) return BFSC_ERR_CUDA;
    *h_n_ids = res[0];
    return BFSC_OK;
}
