// nf_noalloc.cu — nf_aggregate_bucket_noalloc (include/nf.h): the fused per-bucket call for callers that may not
// allocate where they call it (CUDA graph capture, serving loops, harnesses that forbid cudaMalloc). The fused
// kernel's direction workspace is the file-scope device array below instead of a caller buffer; everything else
// is nf_aggregate_bucket, unchanged. No cudaMalloc / cudaFree / allocating routine is called here or below.
//
// g_noalloc_dirs is NF_NOALLOC_WORKSPACE_BYTES (16 MiB) of every GPU that loads libnf.so, held until the
// process exits. In HOST code the name `g_noalloc_dirs` is only the host-side stand-in of the symbol, not a device
// address: the address the kernel is given comes from cudaGetSymbolAddress, asked once per device with that
// device current (this file), and cached per device index.
//
// All calls on a device share the array and it keeps the last call's bytes. Nothing has to be cleared: pass A
// writes every direction byte that pass B of the same launch reads (one byte per 4 low-bit elements, each low-bit
// tensor padded to whole 32-element words). Calls that overlap on the GPU race on it (nf.h).
#include <mutex>
#include "nf_internal.cuh"

static __device__ __align__(256) unsigned char g_noalloc_dirs[NF_NOALLOC_WORKSPACE_BYTES];

namespace {

constexpr int kMaxDevices = 64;
std::mutex g_noalloc_mutex;
void *g_noalloc_ptr[kMaxDevices] = {};   // device address of g_noalloc_dirs on device i, 0 = not looked up yet

// device address of the scratch array on the current device (looked up on the device's first call)
int noalloc_workspace(void **ws) {
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kMaxDevices) return NF_ERR_CUDA;
    std::lock_guard<std::mutex> lock(g_noalloc_mutex);
    if (!g_noalloc_ptr[dev]) {
        void *ptr = nullptr;
        if (cudaGetSymbolAddress(&ptr, g_noalloc_dirs) != cudaSuccess || !ptr) {
            (void)cudaGetLastError();
            return NF_ERR_CUDA;
        }
        g_noalloc_ptr[dev] = ptr;
    }
    *ws = g_noalloc_ptr[dev];
    return NF_OK;
}

}  // namespace

extern "C" int nf_aggregate_bucket_noalloc(const float *g, int64_t worker_stride, int W, int64_t n,
                                           const int64_t *off, const int64_t *len, const uint8_t *elig, int T,
                                           nf_state state, int mode, const float *tau, int margin, float alpha,
                                           uint8_t *route, int64_t *woff, int64_t *summary,
                                           uint32_t *P, uint32_t *N, int64_t plane_stride,
                                           double *abs_sum, double *sumsq, uint64_t *nan_cnt, uint64_t *inf_cnt,
                                           float *out, float *scale_out,
                                           void *plan, size_t plan_bytes, nf_stream stream) {
    // ranges first (nf_aggregate_bucket repeats them), so that "too large" is only said of a bucket that is otherwise valid in size
    if (W < 1 || W > 255 || T < 0 || T > NF_MAX_TENSORS || n < 0 || n > ((int64_t)1 << 40)) return NF_ERR_RANGE;
    if (nf_workspace_bytes(T, n) > NF_NOALLOC_WORKSPACE_BYTES) return NF_ERR_TOO_LARGE;
    void *ws = nullptr;
    const int rc = noalloc_workspace(&ws);
    if (rc != NF_OK) return rc;
    return nf_aggregate_bucket(g, worker_stride, W, n, off, len, elig, T, state, mode, tau, margin, alpha, route, woff,
                               summary, P, N, plane_stride, abs_sum, sumsq, nan_cnt, inf_cnt, out, scale_out, plan,
                               plan_bytes, ws, NF_NOALLOC_WORKSPACE_BYTES, stream);
}
