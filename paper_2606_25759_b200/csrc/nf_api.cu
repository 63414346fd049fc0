// nf_api.cu — the extern "C" entry points declared in include/nf.h: argument checks that can be
// made on the host, then kernel launches on the caller's stream. No allocation, no sync.
#include "nf_internal.cuh"

using namespace nf;

namespace {

unsigned g_trace_calls = 0;
unsigned long long *g_trace = nullptr;   // debug (nf_debug_trace, single-threaded use): per-CTA time stamps of the fused kernel
inline bool misaligned16(const void *p) { return (reinterpret_cast<uintptr_t>(p) & 15u) != 0; }
inline int cuda_rc(cudaError_t e) { return e == cudaSuccess ? NF_OK : NF_ERR_CUDA; }

int check_common(int W, int64_t n, int T) {
    if (W < 1 || W > 255) return NF_ERR_RANGE;
    if (T < 0 || T > NF_MAX_TENSORS) return NF_ERR_RANGE;
    if (n < 0 || n > ((int64_t)1 << 40)) return NF_ERR_RANGE;
    return NF_OK;
}

}  // namespace

extern "C" {

const char *nf_status_string(int status) {
    switch (status) {
        case NF_OK: return "NF_OK";
        case NF_ERR_ARG: return "NF_ERR_ARG: bad argument or bucket layout";
        case NF_ERR_ALIGN: return "NF_ERR_ALIGN: base pointer not 16-byte aligned";
        case NF_ERR_RANGE: return "NF_ERR_RANGE: W, margin, T or n out of range";
        case NF_ERR_CUDA: return "NF_ERR_CUDA: CUDA runtime / launch failure";
        case NF_ERR_TOO_LARGE: return "NF_ERR_TOO_LARGE: bucket needs more scratch than the static NF_NOALLOC_WORKSPACE_BYTES array holds";
        default: return "unknown nf_status";
    }
}

int nf_version(void) { return 200; }

size_t nf_plan_bytes(int T, int R) {
    if (T < 0) T = 0;
    if (R < 1) R = 1;
    return plan_bytes_for(T, R);
}

size_t nf_workspace_bytes(int T, int64_t n) {
    if (T < 0) T = 0;
    if (n < 0) n = 0;
    // one byte per 4 low-bit elements, each L tensor padded to a 32-element word: (n/32 + T) * 8
    return align_up((size_t)(n / 32 + T + 1) * 8, 256);
}

int nf_route_bucket(const int64_t *off, const int64_t *len, const uint8_t *elig, int T, int64_t n,
                    nf_state state, uint8_t *route, int64_t *woff, int64_t *summary,
                    void *plan, size_t plan_bytes, nf_stream stream) {
    int rc = check_common(1, n, T);
    if (rc != NF_OK) return rc;
    if (!summary || !plan || plan_bytes < nf_plan_bytes(T, 1)) return NF_ERR_ARG;
    if (T > 0 && (!off || !len || !elig || !route || !woff)) return NF_ERR_ARG;
    if (misaligned16(plan)) return NF_ERR_ALIGN;
    return cuda_rc(launch_route(off, len, elig, T, n, state, route, woff, summary, plan, plan_bytes, 0, 1,
                                (cudaStream_t)stream));
}

int nf_sign_pack(const float *g, int64_t worker_stride, int W, int64_t n,
                 const int64_t *off, const int64_t *len, const uint8_t *route, const int64_t *woff,
                 int T, int mode, const float *tau,
                 uint32_t *P, uint32_t *N, int64_t plane_stride, double *abs_sum,
                 void *plan, nf_stream stream) {
    int rc = check_common(W, n, T);
    if (rc != NF_OK) return rc;
    if (mode != NF_MODE_GBINARY && mode != NF_MODE_GTERNARY) return NF_ERR_ARG;
    if (!plan || !abs_sum || worker_stride < n || plane_stride < 0) return NF_ERR_ARG;
    if (T > 0 && (!g || !off || !len || !route || !woff || !P)) return NF_ERR_ARG;
    if (mode == NF_MODE_GTERNARY && T > 0 && !N) return NF_ERR_ARG;
    if (misaligned16(g) || misaligned16(P) || misaligned16(N) || misaligned16(plan)) return NF_ERR_ALIGN;
    cudaStream_t s = (cudaStream_t)stream;
    if (T == 0) return NF_OK;
    StreamParams p{};
    p.g = g; p.worker_stride = worker_stride; p.W = W; p.T = T;
    p.off = off; p.len = len; p.route = route; p.woff = woff;
    p.ternary = (mode == NF_MODE_GTERNARY); p.tau = tau;
    p.P = P; p.N = N; p.plane_stride = plane_stride; p.abs_sum = abs_sum; p.plan = plan;
    return cuda_rc(launch_stream(kFPack, p, n, s));
}

int nf_sign_count_reduce(const uint32_t *P, const uint32_t *N, int64_t plane_stride, int W, int64_t n,
                         const int64_t *off, const int64_t *len, const uint8_t *route,
                         const int64_t *woff, int T, int mode, int margin, const double *abs_sum,
                         float *out, uint8_t *cpos, uint8_t *cneg, float *scale_out,
                         void *plan, nf_stream stream) {
    int rc = check_common(W, n, T);
    if (rc != NF_OK) return rc;
    if (margin < 0 || margin > 255) return NF_ERR_RANGE;
    if (mode != NF_MODE_GBINARY && mode != NF_MODE_GTERNARY) return NF_ERR_ARG;
    if (!plan || plane_stride < 0) return NF_ERR_ARG;
    if (T > 0 && (!P || !off || !len || !route || !woff || !abs_sum || !out)) return NF_ERR_ARG;
    if (mode == NF_MODE_GTERNARY && T > 0 && !N) return NF_ERR_ARG;
    if (misaligned16(P) || misaligned16(N) || misaligned16(out) || misaligned16(plan)) return NF_ERR_ALIGN;
    if (T == 0) return NF_OK;
    ReduceParams p{};
    p.P = P; p.N = N; p.plane_stride = plane_stride; p.W = W; p.T = T;
    p.off = off; p.len = len; p.route = route; p.woff = woff;
    p.ternary = (mode == NF_MODE_GTERNARY); p.margin = margin; p.abs_sum = abs_sum;
    p.out = out; p.cpos = cpos; p.cneg = cneg; p.scale_out = scale_out; p.plan = plan;
    return cuda_rc(launch_count_reduce(p, n, (cudaStream_t)stream));
}

int nf_count_planes(int Wg) {
    if (Wg < 1 || Wg > 255) return NF_ERR_RANGE;
    int B = 0;
    while ((1 << B) <= Wg) ++B;
    return B;
}

int nf_partial_count(const uint32_t *P, const uint32_t *N, int64_t plane_stride, int Wg, int64_t Wd, int mode,
                     int B, uint32_t *cnt_pos, uint32_t *cnt_neg, int64_t count_stride, nf_stream stream) {
    if (Wg < 1 || Wg > 255 || B < 1 || B > 8 || (1 << B) <= Wg) return NF_ERR_RANGE;
    if (Wd < 0 || Wd > ((int64_t)1 << 35)) return NF_ERR_RANGE;
    if (mode != NF_MODE_GBINARY && mode != NF_MODE_GTERNARY) return NF_ERR_ARG;
    if (plane_stride < Wd || count_stride < Wd) return NF_ERR_ARG;
    if (Wd > 0 && (!P || !cnt_pos)) return NF_ERR_ARG;
    if (mode == NF_MODE_GTERNARY && Wd > 0 && (!N || !cnt_neg)) return NF_ERR_ARG;
    if (misaligned16(P) || misaligned16(N) || misaligned16(cnt_pos) || misaligned16(cnt_neg)) return NF_ERR_ALIGN;
    return cuda_rc(launch_partial_count(P, N, plane_stride, Wg, Wd, mode == NF_MODE_GTERNARY, B, cnt_pos, cnt_neg,
                                        count_stride, (cudaStream_t)stream));
}

int nf_partial_count_merge(const uint32_t *cnt_pos, const uint32_t *cnt_neg, int64_t count_stride, int G, int B,
                           int W, int64_t n, const int64_t *off, const int64_t *len, const uint8_t *route,
                           const int64_t *woff, int T, int mode, int margin, const double *abs_sum,
                           float *out, uint8_t *cpos, uint8_t *cneg, float *scale_out, void *plan,
                           nf_stream stream) {
    int rc = check_common(W, n, T);
    if (rc != NF_OK) return rc;
    if (margin < 0 || margin > 255 || G < 1 || G > W || B < 1 || B > 8) return NF_ERR_RANGE;
    if (mode != NF_MODE_GBINARY && mode != NF_MODE_GTERNARY) return NF_ERR_ARG;
    if (!plan || count_stride < 0) return NF_ERR_ARG;
    if (T > 0 && (!cnt_pos || !off || !len || !route || !woff || !abs_sum || !out)) return NF_ERR_ARG;
    if (mode == NF_MODE_GTERNARY && T > 0 && !cnt_neg) return NF_ERR_ARG;
    if (misaligned16(cnt_pos) || misaligned16(cnt_neg) || misaligned16(out) || misaligned16(plan)) return NF_ERR_ALIGN;
    if (T == 0) return NF_OK;
    ReduceParams p{};
    p.cnt_pos = cnt_pos; p.cnt_neg = cnt_neg; p.count_stride = count_stride; p.G = G; p.B = B;
    p.W = W; p.T = T; p.off = off; p.len = len; p.route = route; p.woff = woff;
    p.ternary = (mode == NF_MODE_GTERNARY); p.margin = margin; p.abs_sum = abs_sum;
    p.out = out; p.cpos = cpos; p.cneg = cneg; p.scale_out = scale_out; p.plan = plan;
    return cuda_rc(launch_count_reduce(p, n, (cudaStream_t)stream));
}

int nf_stock_packed_sign(const uint32_t *P, const uint32_t *N, int64_t plane_stride, int W, int64_t n,
                         const int64_t *off, const int64_t *len, const uint8_t *route, const int64_t *woff, int T,
                         int mode, int margin, const double *abs_sum, uint32_t *recvP, uint32_t *recvN,
                         float *out, int64_t out_stride, void *plan, nf_stream stream) {
    int rc = check_common(W, n, T);
    if (rc != NF_OK) return rc;
    if (margin < 0 || margin > 255) return NF_ERR_RANGE;
    if (mode != NF_MODE_GBINARY && mode != NF_MODE_GTERNARY) return NF_ERR_ARG;
    if (!plan || plane_stride < 0 || out_stride < n || (out_stride & 3)) return NF_ERR_ARG;
    if (T > 0 && (!P || !recvP || !off || !len || !route || !woff || !abs_sum || !out)) return NF_ERR_ARG;
    if (mode == NF_MODE_GTERNARY && T > 0 && (!N || !recvN)) return NF_ERR_ARG;
    if (misaligned16(P) || misaligned16(N) || misaligned16(recvP) || misaligned16(recvN) || misaligned16(out) ||
        misaligned16(plan) || (plane_stride & 3))
        return NF_ERR_ALIGN;
    if (T == 0) return NF_OK;
    cudaStream_t s = (cudaStream_t)stream;
    const size_t plane_words = (size_t)W * (size_t)plane_stride;
    for (int r = 0; r < W; ++r) {
        // (1) all-gather: replica r receives every worker's packed planes
        uint32_t *rp = recvP + (size_t)r * plane_words, *rn = recvN ? recvN + (size_t)r * plane_words : nullptr;
        if (plane_words > 0) {
            if (cudaMemcpyAsync(rp, P, plane_words * 4, cudaMemcpyDeviceToDevice, s) != cudaSuccess) return NF_ERR_CUDA;
            if (mode == NF_MODE_GTERNARY &&
                cudaMemcpyAsync(rn, N, plane_words * 4, cudaMemcpyDeviceToDevice, s) != cudaSuccess)
                return NF_ERR_CUDA;
        }
        // (2) local unpack-and-count over the received streams
        ReduceParams p{};
        p.P = rp; p.N = rn; p.plane_stride = plane_stride; p.W = W; p.T = T;
        p.off = off; p.len = len; p.route = route; p.woff = woff;
        p.ternary = (mode == NF_MODE_GTERNARY); p.margin = margin; p.abs_sum = abs_sum;
        p.out = out + (size_t)r * (size_t)out_stride; p.plan = plan;
        if (launch_count_reduce(p, n, s) != cudaSuccess) return NF_ERR_CUDA;
    }
    return NF_OK;
}

int nf_fp32_reduce(const float *g, int64_t worker_stride, int W, int64_t n,
                   const int64_t *off, const int64_t *len, const uint8_t *route, int T,
                   float alpha, float *out, void *plan, nf_stream stream) {
    int rc = check_common(W, n, T);
    if (rc != NF_OK) return rc;
    if (!plan || worker_stride < n) return NF_ERR_ARG;
    if (T > 0 && (!g || !off || !len || !route || !out)) return NF_ERR_ARG;
    if (misaligned16(g) || misaligned16(out) || misaligned16(plan)) return NF_ERR_ALIGN;
    if (T == 0) return NF_OK;
    StreamParams p{};
    p.g = g; p.worker_stride = worker_stride; p.W = W; p.T = T;
    p.off = off; p.len = len; p.route = route; p.alpha = alpha; p.out = out; p.plan = plan;
    return cuda_rc(launch_stream(kFFp32, p, n, (cudaStream_t)stream));
}

int nf_health_stats(const float *x, int64_t replica_stride, int R, int64_t n,
                    const int64_t *off, const int64_t *len, int T,
                    double *sumsq, uint64_t *nan_cnt, uint64_t *inf_cnt,
                    void *plan, nf_stream stream) {
    if (R < 1 || R > (1 << 20)) return NF_ERR_RANGE;
    int rc = check_common(1, n, T);
    if (rc != NF_OK) return rc;
    if (!plan || replica_stride < n || !sumsq || !nan_cnt || !inf_cnt) return NF_ERR_ARG;
    if (T > 0 && (!x || !off || !len)) return NF_ERR_ARG;
    if (misaligned16(x) || misaligned16(plan)) return NF_ERR_ALIGN;
    if (T == 0) return NF_OK;
    cudaStream_t s = (cudaStream_t)stream;
    StreamParams p{};
    p.g = x; p.worker_stride = replica_stride; p.W = R; p.T = T;
    p.off = off; p.len = len; p.route = nullptr;
    p.sumsq = sumsq; p.nan_cnt = (unsigned long long *)nan_cnt; p.inf_cnt = (unsigned long long *)inf_cnt;
    p.plan = plan;
    return cuda_rc(launch_stream(kFHealth, p, n, s));
}

}  // extern "C"

namespace {

struct Chain {                 // how a bucket's kernel is linked to its neighbours inside nf_aggregate_step
    const nf_bucket *prev = nullptr;
    const nf_bucket *pp = nullptr;   // the bucket before prev, when prev's kernel was chained to it
    const void *prev_dirs = nullptr;
    int prev_W = 0;
    bool chained = false, next_chained = false;
};

int check_bucket(const nf_bucket &b, int W, int mode, int margin, const void *workspace, size_t workspace_bytes) {
    int rc = check_common(W, b.n, b.T);
    if (rc != NF_OK) return rc;
    if (margin < 0 || margin > 255) return NF_ERR_RANGE;
    if (mode != NF_MODE_GBINARY && mode != NF_MODE_GTERNARY) return NF_ERR_ARG;
    if (!b.summary || !b.plan || b.plan_bytes < nf_plan_bytes(b.T, W)) return NF_ERR_ARG;
    if (!workspace || workspace_bytes < nf_workspace_bytes(b.T, b.n)) return NF_ERR_ARG;
    if (b.worker_stride < b.n || b.plane_stride < 0 || !b.abs_sum) return NF_ERR_ARG;
    if (b.T > 0 && (!b.g || !b.off || !b.len || !b.elig || !b.route || !b.woff || !b.out)) return NF_ERR_ARG;
    if (b.P && mode == NF_MODE_GTERNARY && !b.N) return NF_ERR_ARG;
    const bool health = b.sumsq || b.nan_cnt || b.inf_cnt;
    if (health && !(b.sumsq && b.nan_cnt && b.inf_cnt)) return NF_ERR_ARG;
    if (misaligned16(b.g) || misaligned16(b.out) || misaligned16(b.P) || misaligned16(b.N) ||
        misaligned16(b.plan) || misaligned16(workspace))
        return NF_ERR_ALIGN;
    return NF_OK;
}

// one bucket through the fused path (arguments already checked)
int launch_bucket(const nf_bucket &b, int W, nf_state state, int mode, int margin, float alpha, void *workspace,
                  const Chain &ch, cudaStream_t s) {
    const int T = b.T;
    // a1: inside the fused kernel for buckets of up to kMetaCap tensors (one launch per bucket), else by the
    // route kernel first (PDL-chained). An empty bucket only gets its summary written.
    const bool inkernel = T > 0 && T <= kMetaCap;
    if (!inkernel) {
        if (launch_route(b.off, b.len, b.elig, T, b.n, state, b.route, b.woff, b.summary, b.plan, b.plan_bytes, 1, 0, s) !=
            cudaSuccess)
            return NF_ERR_CUDA;
        if (T == 0) return NF_OK;
    }
    // one read of the W x n gradients: pass A + pass B in one persistent kernel (nf_fused.cu)
    StreamParams p{};
    p.g = b.g; p.worker_stride = b.worker_stride; p.W = W; p.T = T;
    p.off = b.off; p.len = b.len; p.route = b.route; p.woff = b.woff;
    p.ternary = (mode == NF_MODE_GTERNARY); p.tau = b.tau; p.margin = margin; p.alpha = alpha;
    p.P = b.P; p.N = b.N; p.plane_stride = b.plane_stride;
    p.abs_sum = b.abs_sum; p.sumsq = b.sumsq;
    p.nan_cnt = (unsigned long long *)b.nan_cnt; p.inf_cnt = (unsigned long long *)b.inf_cnt;
    p.out = b.out; p.dirs = (uint8_t *)workspace; p.plan = b.plan;
    p.scale_out = b.scale_out;
    p.trace = g_trace ? g_trace + (size_t)(g_trace_calls++ & 1) * 256 * 16 : nullptr;
    p.inkernel_route = inkernel ? 1 : 0;
    p.elig = b.elig; p.st = state; p.n = b.n; p.route_w = b.route; p.woff_w = b.woff; p.summary = b.summary;
    p.acc_slots = (int64_t)((b.plan_bytes - plan_layout(T).acc) / (sizeof(unsigned long long) * kAccWords));
    p.chained = ch.chained ? 1 : 0;
    p.next_chained = ch.next_chained ? 1 : 0;
    p.defer_tail = ch.next_chained ? 1 : 0;
    if (ch.chained) {
        p.prev_plan = ch.prev->plan; p.prev_T = ch.prev->T; p.prev_W = ch.prev_W;
        if (ch.pp) { p.pp_plan = ch.pp->plan; p.pp_T = ch.pp->T; p.pp_W = ch.prev_W; }
        p.prev_off = ch.prev->off; p.prev_len = ch.prev->len; p.prev_woff = ch.prev->woff;
        p.prev_route = ch.prev->route; p.prev_dirs = (const uint8_t *)ch.prev_dirs; p.prev_out = ch.prev->out;
    }
    const bool health = b.sumsq != nullptr;
    return cuda_rc(launch_fused_passA(health, p, b.n, s));
}

}  // namespace

extern "C" {

int nf_aggregate_bucket(const float *g, int64_t worker_stride, int W, int64_t n,
                        const int64_t *off, const int64_t *len, const uint8_t *elig, int T,
                        nf_state state, int mode, const float *tau, int margin, float alpha,
                        uint8_t *route, int64_t *woff, int64_t *summary,
                        uint32_t *P, uint32_t *N, int64_t plane_stride,
                        double *abs_sum, double *sumsq, uint64_t *nan_cnt, uint64_t *inf_cnt,
                        float *out, float *scale_out,
                        void *plan, size_t plan_bytes, void *workspace, size_t workspace_bytes,
                        nf_stream stream) {
    nf_bucket b{};
    b.g = g; b.worker_stride = worker_stride; b.n = n; b.off = off; b.len = len; b.elig = elig; b.T = T; b.tau = tau;
    b.route = route; b.woff = woff; b.summary = summary; b.P = P; b.N = N; b.plane_stride = plane_stride;
    b.abs_sum = abs_sum; b.sumsq = sumsq; b.nan_cnt = nan_cnt; b.inf_cnt = inf_cnt; b.out = out; b.scale_out = scale_out;
    b.plan = plan; b.plan_bytes = plan_bytes;
    const int rc = check_bucket(b, W, mode, margin, workspace, workspace_bytes);
    if (rc != NF_OK) return rc;
    return launch_bucket(b, W, state, mode, margin, alpha, workspace, Chain{}, (cudaStream_t)stream);
}

size_t nf_step_workspace_bytes(const nf_bucket *buckets, int nb) {
    size_t total = 0;
    for (int i = 0; buckets && i < nb; ++i) total += nf_workspace_bytes(buckets[i].T, buckets[i].n);
    return total > 0 ? total : nf_workspace_bytes(0, 0);
}

int nf_aggregate_step(const nf_bucket *buckets, int nb, int W, nf_state state, int mode, int margin, float alpha,
                      void *workspace, size_t workspace_bytes, nf_stream stream) {
    if (nb < 0 || (nb > 0 && !buckets)) return NF_ERR_ARG;
    if (!workspace || workspace_bytes < nf_step_workspace_bytes(buckets, nb)) return NF_ERR_ARG;
    // everything is checked before anything is launched
    for (int i = 0; i < nb; ++i) {
        const int rc = check_bucket(buckets[i], W, mode, margin, workspace, nf_workspace_bytes(buckets[i].T, buckets[i].n));
        if (rc != NF_OK) return rc;
        for (int j = 0; j < i; ++j)
            if (buckets[j].plan == buckets[i].plan || (buckets[i].n > 0 && buckets[j].n > 0 && buckets[j].out == buckets[i].out))
                return NF_ERR_ARG;                            // buckets of a step must not share plans or outputs
    }
    // Every bucket gets its own slice of the workspace: several kernels of the chain can be in flight at once (a
    // small bucket's kernel starts on idle SMs while its predecessors still run), so no slice is ever reused
    // inside a step.
    auto chainable = [&](int i) { return buckets[i].T > 0 && buckets[i].T <= kMetaCap; };
    size_t slice_off = 0, prev_off = 0;
    for (int i = 0; i < nb; ++i) {
        Chain ch;
        ch.chained = i > 0 && chainable(i) && chainable(i - 1);
        ch.next_chained = i + 1 < nb && chainable(i) && chainable(i + 1);
        if (ch.chained) {
            ch.prev = &buckets[i - 1];
            if (i >= 2 && chainable(i - 2)) ch.pp = &buckets[i - 2];      // (kernel i-1 was chained to i-2)
            ch.prev_dirs = (const char *)workspace + prev_off;
            ch.prev_W = W;
        }
        const int rc = launch_bucket(buckets[i], W, state, mode, margin, alpha, (char *)workspace + slice_off, ch,
                                     (cudaStream_t)stream);
        if (rc != NF_OK) return rc;
        prev_off = slice_off;
        slice_off += nf_workspace_bytes(buckets[i].T, buckets[i].n);
    }
    return NF_OK;
}

// debug aid (nf.h): enable (on != 0) allocates a device buffer of 256 x 8 stamps the fused kernel fills;
// with `out` != NULL the stamps are copied to the host (synchronises).
int nf_debug_trace(int on, unsigned long long *out) {
    const size_t bytes = 2 * 256 * 16 * sizeof(unsigned long long);
    if (on && !g_trace) {
        if (cudaMalloc(&g_trace, bytes) != cudaSuccess) return NF_ERR_CUDA;
        cudaMemset(g_trace, 0, bytes);
        g_trace_calls = 0;
    }
    if (out && g_trace && cudaMemcpy(out, g_trace, bytes, cudaMemcpyDeviceToHost) != cudaSuccess) return NF_ERR_CUDA;
    if (!on && g_trace) { cudaFree(g_trace); g_trace = nullptr; }
    return NF_OK;
}

int nf_aggregate_bucket_host(const float *g_host, float *g_dev, int64_t worker_stride, int W,
                             int64_t n, const int64_t *off, const int64_t *len, const uint8_t *elig,
                             int T, nf_state state, int mode, const float *tau, int margin, float alpha,
                             uint8_t *route, int64_t *woff, int64_t *summary,
                             uint32_t *P, uint32_t *N, int64_t plane_stride,
                             double *abs_sum, double *sumsq, uint64_t *nan_cnt, uint64_t *inf_cnt,
                             float *out, float *out_host,
                             void *plan, size_t plan_bytes, void *workspace, size_t workspace_bytes,
                             nf_stream stream) {
    int rc = check_common(W, n, T);
    if (rc != NF_OK) return rc;
    if (!g_host || !g_dev || !out_host || worker_stride < n) return NF_ERR_ARG;
    if (misaligned16(g_dev)) return NF_ERR_ALIGN;
    cudaStream_t s = (cudaStream_t)stream;
    // W rows of n floats, `worker_stride` apart: the last row ends at (W-1)*worker_stride + n
    const size_t count = (size_t)(W - 1) * (size_t)worker_stride + (size_t)n;
    if (n > 0 && cudaMemcpyAsync(g_dev, g_host, sizeof(float) * count, cudaMemcpyHostToDevice, s) != cudaSuccess)
        return NF_ERR_CUDA;
    rc = nf_aggregate_bucket(g_dev, worker_stride, W, n, off, len, elig, T, state, mode, tau, margin,
                             alpha, route, woff, summary, P, N, plane_stride, abs_sum, sumsq, nan_cnt,
                             inf_cnt, out, nullptr, plan, plan_bytes, workspace, workspace_bytes, stream);
    if (rc != NF_OK) return rc;
    if (n > 0 && cudaMemcpyAsync(out_host, out, sizeof(float) * (size_t)n, cudaMemcpyDeviceToHost, s) != cudaSuccess)
        return NF_ERR_CUDA;
    return NF_OK;
}

}  // extern "C"
