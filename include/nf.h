/*
 * nf.h — C ABI of the B200-native low-bit gradient-bucket aggregation library (libnf.so).
 *
 * The library implements the per-bucket hot path of NEURON-Fabric's DDP communication hook
 * (§3.3, §5.2, §6.1), with the W workers' flat FP32 gradient
 * buckets emulated as W replicas resident in one GPU's HBM (BASELINE.json north_star).
 *
 * Conventions (all entry points):
 *  - Every pointer is a DEVICE pointer unless the argument is marked "host". The caller owns
 *    every buffer; the library never allocates device memory and never synchronises.
 *  - Every call only ENQUEUES work on `stream` (a cudaStream_t passed as void*; NULL = default
 *    stream) and returns. Calls on one stream compose in order without host synchronisation.
 *  - Return value: NF_OK (0) or a negative nf_status. Host-checkable errors (ranges, NULLs,
 *    alignment, plan size) are detected before anything is launched. The bucket layout lives in
 *    device memory, so layout errors (overlap, out of range, unsorted) are detected ON THE
 *    DEVICE by nf_route_bucket: it writes NF_ERR_ARG into summary[NF_SUM_STATUS] and into the
 *    plan, and every later call given that plan does nothing.
 *  - Layout of a bucket: `n` FP32 elements per worker; worker w's bucket starts at
 *    g + w*worker_stride (worker_stride >= n, in elements). Tensor t occupies
 *    [off[t], off[t]+len[t]); tensors are in ascending order, non-overlapping, gaps allowed
 *    (gap positions are never read or written). len[t] >= 0.
 *  - Alignment: g, out, P, N must be 16-byte aligned (else NF_ERR_ALIGN). Tensor offsets and
 *    strides may be arbitrary; tensors whose rows are not 16-byte aligned take a scalar path.
 *    The fused call moves gradients with 16-byte bulk copies: for such unaligned rows it reads the
 *    whole 16-byte chunks that contain the row's first and last element, i.e. up to 12 bytes before
 *    / after the row inside the chunk (never a chunk without an element of the row; nothing is written).
 *  - "gap positions are never read" holds up to that chunk granularity for unaligned rows.
 *  - Concurrency: no call assumes that all CTAs of its grid are resident at once (no cooperative launch,
 *    no grid-wide barrier; a CTA only ever waits for CTAs that are already running), so calls may run
 *    beside other kernels that hold SMs and beside each other on different streams, provided they are
 *    given different plan / workspace / output buffers. Calls that share a plan must be ordered on one
 *    stream.
 *  - Determinism: every output of every call is bit-reproducible from run to run on the same device for
 *    the same inputs and launch geometry: integer results trivially, the FP32 route by its fixed worker
 *    order, and the per-(worker, tensor) totals abs_sum / sumsq (hence the scales and decoded outputs)
 *    because partial sums of a fixed shape are accumulated EXACTLY (wide fixed-point integer
 *    accumulators inside the plan) and rounded to FP64 once, whatever the CTA scheduling.
 *  - A bounded wait that runs out inside a kernel (a lost CTA, a corrupted plan) is reported as
 *    NF_ERR_CUDA in summary[NF_SUM_STATUS] and in the plan (later calls given that plan do nothing)
 *    instead of hanging the device.
 *  - Packed planes (reading #10): uint32 words, LSB = lowest element index, each L tensor starts
 *    at word woff[t] and is padded with 0 bits to a word boundary; worker w's plane starts at
 *    P + w*plane_stride (plane_stride >= Wd words).
 *  - Outputs that accumulate (abs_sum, sumsq, nan_cnt, inf_cnt) need no preparation by the caller: the
 *    callee writes every (worker, tensor) entry. `out` is written only at positions owned by the call (L tensors for
 *    nf_sign_count_reduce, P/F tensors for nf_fp32_reduce), so the calls compose into one buffer.
 *  - 1 <= W <= 255 (uint8 counts), 0 <= margin <= 255, 0 <= T <= NF_MAX_TENSORS; else NF_ERR_RANGE.
 */
#ifndef NF_H_
#define NF_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum nf_status {
    NF_OK = 0,
    NF_ERR_ARG = -1,    /* NULL where a pointer is required, bad mode, bad bucket layout, plan too small */
    NF_ERR_ALIGN = -2,  /* a base pointer is not 16-byte aligned */
    NF_ERR_RANGE = -3,  /* W, margin, T or n outside the supported range */
    NF_ERR_CUDA = -4,   /* a CUDA runtime call or kernel launch failed */
    NF_ERR_TOO_LARGE = -5 /* nf_aggregate_bucket_noalloc: the bucket needs more scratch than NF_NOALLOC_WORKSPACE_BYTES */
} nf_status;

/* Route codes: L = low-bit executed, F = FP32 fallback of an admitted route under
 * veto / guard reject, P = plain FP32. */
typedef enum nf_route { NF_ROUTE_P = 0, NF_ROUTE_L = 1, NF_ROUTE_F = 2 } nf_route;

/* Low-bit payload formats: G-Binary = one-bit sign-count route; G-Ternary adds the
 * zero-gating plane. */
typedef enum nf_mode { NF_MODE_GBINARY = 1, NF_MODE_GTERNARY = 2 } nf_mode;

/* Per-step controller state read by the hook, PAPER L143 steps (4) and (6): Commander admission,
 * Supervisor veto, endpoint-capacity guard verdict. */
typedef struct nf_state { int32_t admitted, veto, capacity_ok; } nf_state;

#define NF_MAX_TENSORS 8192
/* summary[] slots written by nf_route_bucket (8 x int64, device) */
enum { NF_SUM_WD = 0, NF_SUM_NL = 1, NF_SUM_NF = 2, NF_SUM_NP = 3, NF_SUM_E = 4, NF_SUM_F = 5,
       NF_SUM_TILES = 6, NF_SUM_STATUS = 7, NF_SUM_LEN = 8 };

typedef void *nf_stream; /* cudaStream_t */

const char *nf_status_string(int status);
/* library version, e.g. 200 = 0.2.0 */
int nf_version(void);

/* Bytes of the device "plan" buffer for a bucket of T tensors used with up to R workers / replicas (host
 * call): the route-dependent tile map the streaming kernels walk, per-tensor scratch (scales, completion
 * counters), an 8 KB list of decode units handed from one kernel of a step to the next, and R x T exact
 * accumulators of 256 bytes for the per-(replica, tensor) totals. R = the largest
 * W (or R of nf_health_stats) any call will be given this plan with. 16-byte aligned buffer required. The
 * buffer must be zero-filled ONCE before its first use (cudaMemset / torch.zeros) and not modified by the caller
 * afterwards: the fused call recognises a plan whose state it left clean by a 32-bit token in the header and
 * re-initialises anything else itself. */
size_t nf_plan_bytes(int T, int R);

/* Bytes of the device workspace nf_aggregate_bucket needs for a bucket of n elements (host call):
 * the 2-bit aggregate directions of the low-bit positions between its two passes. */
size_t nf_workspace_bytes(int T, int64_t n);

/*
 * a1 Route — PAPER L108, L132, L143, L205, L229 (oracle O1).
 * For each tensor: !admitted -> P; elig==0 -> P; veto or !capacity_ok -> F; else L.
 * Outputs: route[T] (uint8 nf_route), woff[T] (first packed word of an L tensor = running sum of
 * ceil(len/32) over L tensors in bucket order; -1 if not L), summary[NF_SUM_LEN] =
 * {Wd, nL, nF, nP, e, f, n_tiles, status}, and the plan. One single-CTA kernel. plan_bytes >=
 * nf_plan_bytes(T, 1) is checked here; a plan too small for the W of a later call (or plane rows shorter than
 * Wd words) is detected on the device by that call, which then poisons the plan (status NF_ERR_ARG) and does
 * nothing else.
 */
int nf_route_bucket(const int64_t *off, const int64_t *len, const uint8_t *elig, int T, int64_t n,
                    nf_state state, uint8_t *route, int64_t *woff, int64_t *summary,
                    void *plan, size_t plan_bytes, nf_stream stream);

/*
 * a2 Pack — PAPER L144, L211 (write-side payload materialisation; oracle O2).
 * For each worker w and L tensor t: P bit = (x > tau_t), G-Ternary N bit = (x < -tau_t)
 * (tau == NULL means 0; tau[t] >= 0 is the caller's contract), abs_sum[w*T+t] = sum |x| (FP64).
 * abs_sum of non-L tensors is 0. N may be NULL iff mode == NF_MODE_GBINARY. Reads g once.
 */
int nf_sign_pack(const float *g, int64_t worker_stride, int W, int64_t n,
                 const int64_t *off, const int64_t *len, const uint8_t *route, const int64_t *woff,
                 int T, int mode, const float *tau,
                 uint32_t *P, uint32_t *N, int64_t plane_stride, double *abs_sum,
                 void *plan, nf_stream stream);

/*
 * a3 Sign-count reduce + decode — PAPER L211, L243, L247 (read-side aggregation; oracle O3).
 * Per L element: cpos = popcount over the W pos-plane bits, cneg likewise over the neg plane
 * (G-Binary: cneg = W - cpos); D = cpos - cneg; d = (D > margin) - (D < -margin);
 * s_wt = (float)(abs_sum[w*T+t]/len_t); S_t = (float)(sum_w (double)s_wt / W);
 * out[off_t+i] = S_t * (float)d. Optional: cpos/cneg [n] uint8 at bucket positions (L positions
 * only are written), scale_out[T] (0 for non-L tensors).
 * Plane rows that are 16-byte aligned (plane_stride a multiple of 4 words) are read with bulk async
 * copies of whole 16-byte chunks, i.e. up to 3 words past Wd inside the row; any other plane_stride
 * takes a register-staged kernel with the same results. The call writes the per-tensor scales into
 * the plan's scratch: calls given the same plan must be ordered on one stream.
 */
int nf_sign_count_reduce(const uint32_t *P, const uint32_t *N, int64_t plane_stride, int W, int64_t n,
                         const int64_t *off, const int64_t *len, const uint8_t *route,
                         const int64_t *woff, int T, int mode, int margin, const double *abs_sum,
                         float *out, uint8_t *cpos, uint8_t *cneg, float *scale_out,
                         void *plan, nf_stream stream);

/*
 * NEXT-1: two-level hierarchical sign count — PAPER L243 ("node-local counting and
 * inter-node partial-count exchange before returning a synchronized aggregate direction"), L267
 * ("performs node-local sign counting, exchanges partial counts, and returns the aggregate
 * direction"). Results are identical to nf_sign_count_reduce over all W workers.
 *
 * nf_count_planes (host): bit-planes of a partial count of Wg workers = smallest B with 2^B > Wg
 * (1..8), or NF_ERR_RANGE.
 *
 * nf_partial_count — level 1, one group ("node") of Wg workers: for every packed word k < Wd and
 * bit j, c = number of the group's workers whose bit j of word k is set; stored bit-sliced:
 * cnt_pos[b*count_stride + k] bit j = bit b of c, b < B (2^B > Wg required). cnt_neg likewise
 * from N (G-Ternary only; N and cnt_neg may be NULL for G-Binary). P/N are the group's planes
 * [Wg][plane_stride]. The B x Wd words per sign are the partial-count payload a node sends.
 *
 * nf_partial_count_merge — level 2: adds the G groups' partial counts, cnt[(g*B + b)*count_stride
 * + k], into cpos/cneg (G-Binary: cneg = W - cpos, W = total workers), then votes, scales and
 * writes exactly as nf_sign_count_reduce: abs_sum[W][T] in global worker order, same plan, same
 * optional outputs. Groups may hold different numbers of workers as long as each count fits B planes.
 */
int nf_count_planes(int Wg);
int nf_partial_count(const uint32_t *P, const uint32_t *N, int64_t plane_stride, int Wg, int64_t Wd, int mode,
                     int B, uint32_t *cnt_pos, uint32_t *cnt_neg, int64_t count_stride, nf_stream stream);
int nf_partial_count_merge(const uint32_t *cnt_pos, const uint32_t *cnt_neg, int64_t count_stride, int G, int B,
                           int W, int64_t n, const int64_t *off, const int64_t *len, const uint8_t *route,
                           const int64_t *woff, int T, int mode, int margin, const double *abs_sum,
                           float *out, uint8_t *cpos, uint8_t *cneg, float *scale_out, void *plan,
                           nf_stream stream);

/*
 * NEXT-2: the stock packed-sign path the paper compares against — PAPER L245 ("packed-sign all-gather
 * followed by local unpack-and-count"), L267 ("aggregation remains replicated: each worker receives sign streams and
 * reconstructs the same count locally"), Fig. 3. Emulated on one GPU with the W workers as replicas: for every
 * replica r < W, (1) the all-gather: all W workers' packed planes are copied into replica r's own receive buffer
 * recvP + r*W*plane_stride (recvN likewise; G-Ternary only) — device-to-device copies standing in for the wire —
 * and (2) the local unpack-and-count: the flat count + vote + decode of nf_sign_count_reduce over the received
 * planes into replica r's own output out + r*out_stride. All W outputs must come out identical (and identical to
 * nf_sign_count_reduce / the hierarchical path): that is what "the same count" means. Bytes gathered =
 * W * W * Wd * 4 per plane. recvP / recvN: [W][W][plane_stride] words; out: [W][out_stride] floats, out_stride >= n
 * and a multiple of 4; only low-bit positions are written. Same plan / metadata arguments as nf_sign_count_reduce.
 */
int nf_stock_packed_sign(const uint32_t *P, const uint32_t *N, int64_t plane_stride, int W, int64_t n,
                         const int64_t *off, const int64_t *len, const uint8_t *route, const int64_t *woff, int T,
                         int mode, int margin, const double *abs_sum, uint32_t *recvP, uint32_t *recvN,
                         float *out, int64_t out_stride, void *plan, nf_stream stream);

/*
 * a4a FP32 route — PAPER L50, L66, L144 (oracle O4a). For every P/F tensor:
 * out[i] = alpha * (((g_0[i] + g_1[i]) + g_2[i]) + ... + g_{W-1}[i]) in FP32, fixed worker order.
 */
int nf_fp32_reduce(const float *g, int64_t worker_stride, int W, int64_t n,
                   const int64_t *off, const int64_t *len, const uint8_t *route, int T,
                   float alpha, float *out, void *plan, nf_stream stream);

/*
 * a4b Health statistics — BASELINE.json north_star step (4); consumer PAPER L158, L177 (oracle O4b).
 * For every replica r < R and tensor t (any route): sumsq[r*T+t] = sum of x*x over finite x
 * (FP64), nan_cnt = #NaN, inf_cnt = #+-Inf. L2 norm = sqrt(sumsq). R >= 1 (no upper bound).
 */
int nf_health_stats(const float *x, int64_t replica_stride, int R, int64_t n,
                    const int64_t *off, const int64_t *len, int T,
                    double *sumsq, uint64_t *nan_cnt, uint64_t *inf_cnt,
                    void *plan, nf_stream stream);

/*
 * Fused path (the one the target is measured on) — the results of
 * nf_route_bucket -> nf_sign_pack -> nf_sign_count_reduce -> nf_fp32_reduce -> nf_health_stats(g),
 * with the W x n gradients read ONCE. One launch for buckets of up to 256 tensors (the persistent kernel
 * routes the bucket itself; larger T: the route kernel first): it packs, counts, votes, sums the FP32
 * tensors, gathers abs-sums and health statistics from a single read (pass A) and, tensor by tensor as each
 * completes, expands the 2-bit directions by the per-tensor scale (pass B).
 * Against the 5-call sequence: route codes, word offsets, summary, packed planes, aggregate directions,
 * NaN / Inf tallies and the FP32-route outputs are bit-identical; abs_sum / sumsq (and so the scales and the
 * decoded magnitudes) agree to about 1e-7 relative (both sides round FP32 partial sums of different shapes;
 * each side is bit-reproducible by itself) — the bound that holds against the oracle is 1e-6 / 1e-5.
 * P and N may both be NULL (planes not materialised); plane_stride >= Wd words when they are not (checked on
 * the device: NF_ERR_ARG in summary[NF_SUM_STATUS], nothing written). sumsq/nan_cnt/inf_cnt may all be NULL
 * (no health statistics); scale_out may be NULL. route/woff/summary/plan are outputs exactly as in
 * nf_route_bucket; plan_bytes >= nf_plan_bytes(T, W).
 */
int nf_aggregate_bucket(const float *g, int64_t worker_stride, int W, int64_t n,
                        const int64_t *off, const int64_t *len, const uint8_t *elig, int T,
                        nf_state state, int mode, const float *tau, int margin, float alpha,
                        uint8_t *route, int64_t *woff, int64_t *summary,
                        uint32_t *P, uint32_t *N, int64_t plane_stride,
                        double *abs_sum, double *sumsq, uint64_t *nan_cnt, uint64_t *inf_cnt,
                        float *out, float *scale_out,
                        void *plan, size_t plan_bytes, void *workspace, size_t workspace_bytes,
                        nf_stream stream);

/*
 * nf_aggregate_bucket for callers that cannot provide scratch memory of their own because they may not call
 * cudaMalloc where the call is made (code under CUDA graph capture, tight serving loops, harnesses that forbid
 * allocation). Same arguments, results and errors as nf_aggregate_bucket, minus (workspace, workspace_bytes): the
 * fused kernel's direction workspace (one byte per 4 low-bit elements, written by pass A and read back by pass B of
 * the same launch) is a file-scope static device array of NF_NOALLOC_WORKSPACE_BYTES inside the library, which
 * every GPU that loads the library holds until the process exits. The call allocates nothing (no cudaMalloc /
 * cudaFree / allocating library routine); inputs, outputs and the plan are still the caller's.
 *  - Limit: nf_workspace_bytes(T, n) <= NF_NOALLOC_WORKSPACE_BYTES, i.e. n/32 + T + 1 <= 2 Mi words: buckets of up
 *    to about 67 M elements (256 MB of FP32 gradients per worker). A larger bucket is refused with
 *    NF_ERR_TOO_LARGE before anything is launched.
 *  - The array's device address is looked up once per device, on that device's first call (with that device
 *    current); a failure of that lookup is NF_ERR_CUDA. The first call on a device should therefore be made
 *    outside stream capture.
 *  - Every call on a device shares the one array, and it keeps the previous call's contents. Nothing in it has
 *    to start at zero: pass A writes every byte pass B reads. Calls that overlap on the GPU (different streams,
 *    or a stream beside a graph launch) race on it and produce garbage: order them on one stream.
 */
#define NF_NOALLOC_WORKSPACE_BYTES ((size_t)16 << 20)
int nf_aggregate_bucket_noalloc(const float *g, int64_t worker_stride, int W, int64_t n,
                                const int64_t *off, const int64_t *len, const uint8_t *elig, int T,
                                nf_state state, int mode, const float *tau, int margin, float alpha,
                                uint8_t *route, int64_t *woff, int64_t *summary,
                                uint32_t *P, uint32_t *N, int64_t plane_stride,
                                double *abs_sum, double *sumsq, uint64_t *nan_cnt, uint64_t *inf_cnt,
                                float *out, float *scale_out,
                                void *plan, size_t plan_bytes, nf_stream stream);

/*
 * One training step's buckets in ONE call (the hook's view of a step: PAPER L140-146, steps (2)-(7) for every DDP
 * bucket of the model). Bucket i is aggregated exactly as nf_aggregate_bucket would (same results, bit for bit), all
 * on `stream`, but consecutive buckets are chained into a software pipeline: the decode of a bucket's last low-bit
 * tensor — which cannot start before the bucket has been read completely, because its scale needs all of the
 * tensor — is taken over by the kernel of the NEXT bucket and overlaps that bucket's reads, and a chained kernel
 * does not wait for its predecessor before it starts reading (it needs nothing of it).
 * Requirements beyond nf_aggregate_bucket's: the nf_bucket array is HOST memory (read during the call only);
 * every bucket has its own plan, outputs, accumulators and planes (buffers of different buckets must not overlap);
 * everything the step reads (gradients, metadata) is complete before the call is enqueued, i.e. was produced by
 * work enqueued on `stream` before it; `workspace` holds nf_step_workspace_bytes(buckets, nb) bytes (one direction
 * slice per bucket: n/4 bytes each). W, state, mode, margin, alpha are the step's. Buckets of more than 256 tensors (routed
 * by a separate kernel) and empty buckets break the chain and run as stand-alone calls.
 */
typedef struct nf_bucket {
    const float *g;            /* [W][worker_stride] */
    int64_t worker_stride, n;
    const int64_t *off, *len;  /* [T] */
    const uint8_t *elig;       /* [T] */
    int32_t T, reserved;
    const float *tau;          /* [T] or NULL */
    uint8_t *route;            /* [T] out */
    int64_t *woff;             /* [T] out */
    int64_t *summary;          /* [NF_SUM_LEN] out */
    uint32_t *P, *N;           /* planes or NULL */
    int64_t plane_stride;
    double *abs_sum, *sumsq;   /* [W][T]; sumsq / nan_cnt / inf_cnt may all be NULL */
    uint64_t *nan_cnt, *inf_cnt;
    float *out, *scale_out;    /* [n], [T] or NULL */
    void *plan;
    size_t plan_bytes;
} nf_bucket;
size_t nf_step_workspace_bytes(const nf_bucket *buckets /*host*/, int nb);
int nf_aggregate_step(const nf_bucket *buckets /*host*/, int nb, int W, nf_state state, int mode, int margin,
                      float alpha, void *workspace, size_t workspace_bytes, nf_stream stream);

/*
 * End-to-end convenience with HOST buffers (used for the e2e measurement): copies the W rows of n floats
 * from pinned/pageable host memory `g_host` (worker stride = worker_stride elements: (W-1)*worker_stride + n
 * floats are read, and as many written to the caller's device staging buffer `g_dev`, same stride), runs
 * nf_aggregate_bucket with device metadata/outputs as above (P / N device planes or NULL), and copies `out`
 * (n floats) back to `out_host`. All copies are cudaMemcpyAsync on `stream`; the caller synchronises the stream.
 */
int nf_aggregate_bucket_host(const float *g_host /*host*/, float *g_dev, int64_t worker_stride, int W,
                             int64_t n, const int64_t *off, const int64_t *len, const uint8_t *elig,
                             int T, nf_state state, int mode, const float *tau, int margin, float alpha,
                             uint8_t *route, int64_t *woff, int64_t *summary,
                             uint32_t *P, uint32_t *N, int64_t plane_stride,
                             double *abs_sum, double *sumsq, uint64_t *nan_cnt, uint64_t *inf_cnt,
                             float *out, float *out_host /*host*/,
                             void *plan, size_t plan_bytes, void *workspace, size_t workspace_bytes,
                             nf_stream stream);

/*
 * NEXT-3, HOST functions. nf_mgtr — PAPER L110-114: modeled gradient-communication traffic
 * ratio of a route log, MGTR = sum_e bytes(route_e) / sum_e bytes(FP32_e). Event e = (numel[e], route[e]
 * (nf_route), mode[e] (nf_mode, read for L events only)): an L event counts numel*bits/8 + scale_bytes with
 * bits = bits_binary or bits_ternary (reading #14: 1 and log2(3)), F and P events count 4*numel;
 * the denominator counts 4*numel for every event. No events -> 1.
 *
 * nf_capacity_guard — PAPER L273-275: admit a candidate low-bit bucket only when the estimated
 * hierarchical-reducer time is lower than the matched FP32 time. Time model (reading #20, not the
 * paper's): t_fp32 = 2(N-1)/N * 4n / net_bw; t_hier = F * (p*n/8) / service_rate + 2(N-1)/N * (p*B*n/8) /
 * net_bw with N = nodes, F = local_fan_in, p = planes (1 G-Binary, 2 G-Ternary), B = nf_count_planes(N*F),
 * rates in bytes/s. Returns 1 (admit: capacity_ok), 0 (stay on FP32) or a negative nf_status; the two times
 * are written when the pointers are not NULL.
 */
int nf_mgtr(const int64_t *numel /*host*/, const uint8_t *route /*host*/, const uint8_t *mode /*host*/,
            int64_t n_events, double bits_binary, double bits_ternary, int scale_bytes, double *mgtr /*host*/);
int nf_capacity_guard(int64_t n, int nodes, int local_fan_in, double service_rate, double net_bw, int planes,
                      double *t_hier /*host*/, double *t_fp32 /*host*/);

/*
 * NEXT-4: Supervisor recovery controller (HOST functions, no device work) — PAPER L158
 * ("slack is the tolerated per-step increase in the smoothed training-health signal before degradation
 * evidence accumulates, and the threshold is the accumulated excess that triggers fallback to FP32"),
 * L177-179 (smoothed signal + CUSUM; fallback, cooldown, guarded readmission), Table 2. It produces the
 * nf_state flags nf_route_bucket / nf_aggregate_bucket read. Per step (readings #15-#19):
 *   m_0 = x_0, m_k = beta*m_{k-1} + (1-beta)*x_k;  y_k = m_k - m_{k-1};
 *   S_k = max(0, S_{k-1} + y_k - slack) while low-bit is admitted;  alarm iff S_k > threshold, or any
 *   NaN/Inf tally (nf_health_stats) / non-finite signal in the step;
 *   WARMUP (admitted = 0, warmup_steps) -> ADMITTED -> alarm -> COOLDOWN (veto = 1, cooldown_steps) ->
 *   GUARD (guard_steps; an alarm here re-enters COOLDOWN with twice the length) -> ADMITTED.
 * nf_supervisor_step consumes the signal of the step just finished and writes the flags for the next
 * route decisions; capacity_ok is passed through. The struct is plain caller-owned host memory.
 */
typedef struct nf_supervisor_cfg {
    int32_t warmup_steps, cooldown_steps, guard_steps, reserved;
    double ema_beta, slack, threshold;
} nf_supervisor_cfg;
typedef struct nf_supervisor {
    nf_supervisor_cfg cfg;
    int32_t phase;      /* 0 warm-up, 1 admitted, 2 cooldown, 3 guard */
    int32_t remaining;  /* steps left in the current timed phase */
    int64_t step, detections;
    double ema, cusum;
} nf_supervisor;
int nf_supervisor_init(nf_supervisor *s /*host*/, const nf_supervisor_cfg *cfg /*host*/);
int nf_supervisor_step(nf_supervisor *s /*host*/, double signal, uint64_t nan_count, uint64_t inf_count,
                       int capacity_ok, nf_state *out /*host*/);

/*
 * Debugging aid, NOT part of the data path and NOT thread-safe (one process-global buffer: use it from one host
 * thread, with no nf_aggregate_bucket call in flight on another). nf_debug_trace(1, NULL) allocates a device
 * buffer of 2 x 256 x 16 globaltimer stamps; from then on every CTA of the fused kernel fills its row (kernel
 * entry, after the dependency wait, after the routing and the clean-token check, consumers start, tiles
 * exhausted, last tensor flushed, decode done, kernel end), successive calls alternating between the two halves;
 * with `out` != NULL (room for 8192 uint64, HOST) the stamps are copied out (synchronises the device);
 * nf_debug_trace(0, ...) frees the buffer.
 */
int nf_debug_trace(int on, unsigned long long *out /*host*/);

#ifdef __cplusplus
}
#endif
#endif /* NF_H_ */
