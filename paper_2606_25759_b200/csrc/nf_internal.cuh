// nf_internal.cuh — internal declarations shared by the libnf translation units (sm_100a).
// Not part of the public ABI (that is include/nf.h).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include "nf.h"

namespace nf {

// ---------------------------------------------------------------------------------------------
// Work decomposition. A *tile* is NF_TILE consecutive elements of ONE tensor, in tensor-relative
// index space (so bit j of packed word k is always lane-aligned, whatever off[t] is). The plan's
// tile_prefix[t] is the exclusive prefix of ceil(len[t]/NF_TILE) over ALL tensors in bucket order;
// persistent CTAs walk tiles blockIdx.x, blockIdx.x+gridDim.x, ... and find the tensor of a tile
// by binary search in tile_prefix (T+1 ints, L1/L2 resident).
// ---------------------------------------------------------------------------------------------
constexpr int kThreads = 256;              // threads per CTA of the streaming kernels
constexpr int kRows = 2;                   // float4 rows per thread per tile
constexpr int kRowElems = kThreads * 4;    // 1024 elements per row
constexpr int kTile = kRows * kRowElems;   // 2048 elements per tile
constexpr int kGroup = 8;                  // workers per register group (8 x 4-bit nibbles = 32 bits)
constexpr uint32_t kPlanMagic = 0x4e46504cu;  // "NFPL"
constexpr int kMetaCap = 256;              // fused kernel: tensors whose metadata lives in shared memory

constexpr int kMaxOrphans = 2048;          // fused path, chained kernels: pass-B units handed on to the next kernel (see orph)

struct PlanHeader {                        // 80 bytes, at plan + 0
    uint32_t magic;
    int32_t status;                        // NF_OK or NF_ERR_ARG (bad layout): later kernels no-op
    int32_t T;
    int32_t nL;
    int64_t n;
    int64_t Wd;                            // total packed words per worker plane
    int32_t n_tiles;
    int32_t finish_count;                  // fused path: CTAs that have finished (the last one resets the state below)
    int32_t unit_cursor;                   // fused path: next pass-B unit (half tile)
    int32_t pad0;
    // fused path: high half = clean_token(T, W) while unit_cursor, finish_count, done[] and acc[] are all zero
    // (the state every call leaves behind), low half = next pass-A scheduling unit (dynamic scheduling over the
    // CTAs). One atomicAdd both takes a unit and proves the state clean.
    unsigned long long sched;
    int64_t acc_slots;                     // capacity of the acc region in (replica, tensor) slots
    int64_t pad1[2];
};
static_assert(sizeof(PlanHeader) == 80, "plan header layout");

// ---------------------------------------------------------------------------------------------
// Deterministic per-(worker, tensor) totals. abs_sum / sumsq are sums over millions of elements gathered by
// many CTAs in an order that depends on the dynamic tile scheduling; floating-point atomics would make the last
// bits (and, rarely, the FP32 scale) depend on that order. Instead every partial (a deterministic FP64 value:
// the fixed-shape sum of one scheduling segment) is added EXACTLY into a wide fixed-point accumulator with
// 64-bit integer atomics (integer addition commutes), and the tensor's last arriver rounds the exact total to
// FP64 once. One slot = 32 x uint64 per (worker, tensor):
//   words  0..9   sum |x|, word k holds the bits [2^(-149 + 32k), 2^(-149 + 32k + 32)) (+ deferred carries):
//                 FP32 magnitudes are multiples of 2^-149 and 2^40 of them stay below 2^168;
//   words 10..28  sum x^2 over finite x, same scheme from 2^-298 (up to 2^296);
//   word  29 / 30 number of NaN / +-Inf elements;  word 31 unused.
// A slot is all-zero between calls: whoever rounds it also clears it.
// ---------------------------------------------------------------------------------------------
constexpr int kAccWords = 32;
constexpr int kAccAbs = 0, kAccAbsWords = 10, kAccAbsBase = -149;
constexpr int kAccSq = 10, kAccSqWords = 19, kAccSqBase = -298;
constexpr int kAccNan = 29, kAccInf = 30;

// One low-bit tensor as step a3 sees it (index li in the plan's list of L tensors): a warp that enters a tensor reads
// this record instead of walking lt_index -> len / off / lt_woff[li], lt_woff[li + 1] (a chain of dependent L2 round trips).
struct __align__(16) LtRec {
    int64_t t;                             // tensor index
    int64_t off, len;                      // bucket offset and length in elements
    int64_t kfirst, kend;                  // packed word range [kfirst, kend)
    int64_t pad;
};
static_assert(sizeof(LtRec) == 48, "LtRec layout");

// Offsets (bytes) of the plan arrays for a bucket of T tensors.
struct PlanLayout {
    size_t tile_prefix;                    // int32 [T+1]
    size_t lt_index;                       // int32 [T]     ids of the L tensors, in order
    size_t lt_woff;                        // int64 [T+1]   woff of the L tensors, lt_woff[nL] = Wd
    size_t lt_rec;                         // LtRec [T]     everything a3 needs of an L tensor in one 48-byte record
    size_t scale;                          // float [T]     per-tensor scale scratch
    size_t done;                           // int32 [T]     tiles of the tensor whose pass-A results are published
    size_t fin;                            // uint64 [T]    fused path: {1, FP32 bits of S_t} once tensor t is finalised, else 0
    size_t orph;                           // int32 [kMaxOrphans]  fused path: pass-B units (+ 1, 0 = none) the decode warps of a
                                           // kernel whose tail is deferred had in hand when their CTAs left: 4 entries per
                                           // (CTA, decode warp), taken and cleared by the next kernel of the step
    size_t acc;                            // uint64 [R*T][kAccWords]  exact accumulators (R = workers / replicas)
    size_t total;                          // without the acc region
};

__host__ __device__ inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

__host__ __device__ inline PlanLayout plan_layout(int T) {
    PlanLayout L;
    size_t o = sizeof(PlanHeader);
    L.tile_prefix = o; o = align_up(o + sizeof(int32_t) * (size_t)(T + 1), 16);
    L.lt_index = o;    o = align_up(o + sizeof(int32_t) * (size_t)(T > 0 ? T : 1), 16);
    L.lt_woff = o;     o = align_up(o + sizeof(int64_t) * (size_t)(T + 1), 16);
    L.lt_rec = o;      o = align_up(o + sizeof(LtRec) * (size_t)(T > 0 ? T : 1), 16);
    L.scale = o;       o = align_up(o + sizeof(float) * (size_t)(T > 0 ? T : 1), 16);
    L.done = o;        o = align_up(o + sizeof(int32_t) * (size_t)(T > 0 ? T : 1), 16);
    L.fin = o;         o = align_up(o + sizeof(unsigned long long) * (size_t)(T > 0 ? T : 1), 16);
    L.orph = o;        o = align_up(o + sizeof(int32_t) * (size_t)kMaxOrphans, 16);
    L.acc = align_up(o, 256);
    L.total = L.acc;
    return L;
}
__host__ __device__ inline size_t plan_bytes_for(int T, int R) {
    return plan_layout(T).acc + sizeof(unsigned long long) * kAccWords * (size_t)(T > 0 ? T : 1) * (size_t)(R > 0 ? R : 1);
}
constexpr uint32_t kInitToken = 0x494e4954u;          // "INIT": a CTA is zeroing the plan's state
__host__ __device__ inline uint32_t clean_token(int T, int W) {
    uint32_t h = (((uint32_t)T << 8) + (uint32_t)W) * 0x9e3779b1u ^ 0x4e46434cu;
    if (h == 0u || h == kInitToken) h ^= 0x5a5a5a5au;
    return h;
}

struct PlanView {
    const PlanHeader *hdr;
    const int32_t *tile_prefix;
    const int32_t *lt_index;
    const int64_t *lt_woff;
    const LtRec *lt_rec;
    float *scale;
    int32_t *done;
    unsigned long long *fin;
    int32_t *orph;
    unsigned long long *acc;
};

__host__ __device__ inline PlanView plan_view(void *plan, int T) {
    PlanLayout L = plan_layout(T);
    char *p = (char *)plan;
    PlanView v;
    v.hdr = (const PlanHeader *)p;
    v.tile_prefix = (const int32_t *)(p + L.tile_prefix);
    v.lt_index = (const int32_t *)(p + L.lt_index);
    v.lt_woff = (const int64_t *)(p + L.lt_woff);
    v.lt_rec = (const LtRec *)(p + L.lt_rec);
    v.scale = (float *)(p + L.scale);
    v.done = (int32_t *)(p + L.done);
    v.fin = (unsigned long long *)(p + L.fin);
    v.orph = (int32_t *)(p + L.orph);
    v.acc = (unsigned long long *)(p + L.acc);
    return v;
}

// ---------------------------------------------------------------------------------------------
// Parameters of the streaming kernel family (pack / fp32 / health / fused pass A).
// ---------------------------------------------------------------------------------------------
struct StreamParams {
    const float *g;            // [W][worker_stride]
    int64_t worker_stride;
    int W;
    int T;
    const int64_t *off;
    const int64_t *len;
    const uint8_t *route;      // NULL for health-only (all tensors processed, no route semantics)
    const int64_t *woff;
    int ternary;               // mode == NF_MODE_GTERNARY
    const float *tau;          // [T] or NULL
    int margin;
    float alpha;
    uint32_t *P;               // may be NULL (planes not materialised)
    uint32_t *N;
    int64_t plane_stride;
    double *abs_sum;           // [W][T]
    double *sumsq;             // [W][T] or NULL
    unsigned long long *nan_cnt;
    unsigned long long *inf_cnt;
    float *out;                // [n]
    float *scale_out;          // [T] or NULL (fused path: the in-kernel decode publishes the scales)
    uint8_t *dirs;             // workspace: one byte per 4 low-bit elements (lo nibble +, hi nibble -)
    void *plan;
    unsigned long long *trace; // debug: per-CTA globaltimer stamps [grid][8], or NULL
    // in-kernel routing (fused path, T <= kMetaCap): step a1 is computed by the fused kernel itself
    int inkernel_route;
    const uint8_t *elig;       // [T]
    nf_state st;
    int64_t n;
    uint8_t *route_w;          // [T] out
    int64_t *woff_w;           // [T] out
    int64_t *summary;          // [NF_SUM_LEN] out
    int64_t acc_slots;         // capacity of the plan's accumulator region, in (replica, tensor) slots
    // chaining (nf_aggregate_step): consecutive buckets of one step form a software pipeline, see nf_fused.cu
    int chained;               // 1: the kernel right before this one on the stream is the fused kernel of `prev`
    int next_chained;          // 1: the kernel right after this one is chained to it
    int defer_tail;            // 1: the next kernel of the step decodes what cannot be decoded before pass A ends
    void *prev_plan;           // previous bucket of the step (its remaining decode units are drained here)
    int prev_T, prev_W;
    void *pp_plan;             // the bucket before that, when it was chained too (else NULL): this kernel resets its
    int pp_T, pp_W;            //   self-cleaning state (everything that used it is complete once kernel i-1 is)
    const int64_t *prev_off, *prev_len, *prev_woff;
    const uint8_t *prev_route;
    const uint8_t *prev_dirs;
    float *prev_out;
};

enum : int {
    kFPack = 1,     // L tiles: bit planes + abs-sum
    kFCount = 2,    // L tiles: per-position counts -> majority direction -> dirs
    kFFp32 = 4,     // non-L tiles: fixed-order FP32 sum -> out
    kFHealth = 8    // all tiles: sum of squares over finite values, NaN / Inf tallies
};

struct ReduceParams {
    const uint32_t *P;
    const uint32_t *N;
    int64_t plane_stride;
    int W;
    int T;
    const int64_t *off;
    const int64_t *len;
    const uint8_t *route;
    const int64_t *woff;
    int ternary;
    int margin;
    const double *abs_sum;
    float *out;
    uint8_t *cpos;
    uint8_t *cneg;
    float *scale_out;
    const uint32_t *cnt_pos;   // NEXT-1 merge: bit-sliced partial counts [(g*B + b)*count_stride + k], else NULL
    const uint32_t *cnt_neg;
    int64_t count_stride;
    int G, B;
    void *plan;
    // NEXT-1 level 1 through the ring kernel (PARTIAL): the B count planes of this group of W workers are the output
    uint32_t *part_pos, *part_neg;
    int64_t part_Wd;           // packed words per plane (no plan, no tensor metadata on this path)
};

// launchers (each returns a cudaError_t from the launch)
cudaError_t launch_route(const int64_t *off, const int64_t *len, const uint8_t *elig, int T, int64_t n,
                         nf_state st, uint8_t *route, int64_t *woff, int64_t *summary, void *plan, size_t plan_bytes,
                         int pdl, int zero_acc, cudaStream_t s);
cudaError_t launch_stream(int flags, const StreamParams &p, int64_t n, cudaStream_t s);
cudaError_t launch_fused_passA(bool health, const StreamParams &p, int64_t n, cudaStream_t s);
cudaError_t launch_count_reduce(const ReduceParams &p, int64_t n, cudaStream_t s);
cudaError_t launch_partial_count(const uint32_t *P, const uint32_t *N, int64_t plane_stride, int Wg, int64_t Wd,
                                 int ternary, int B, uint32_t *cnt_pos, uint32_t *cnt_neg, int64_t count_stride,
                                 cudaStream_t s);
int device_sm_count();


// ---------------------------------------------------------------------------------------------
// Programmatic dependent launch (PDL): the kernels of one nf_aggregate_bucket call (and of
// back-to-back calls) are chained so that a kernel's launch latency and prologue overlap the tail
// of its predecessor. Every kernel executes pdl_wait() before touching global memory (a no-op
// when it was launched without the attribute), so completion is transitive along the chain.
// ---------------------------------------------------------------------------------------------
#ifdef __CUDACC__
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

template <typename... KArgs, typename... Args>
inline cudaError_t launch_kernel_ex(void (*kernel)(KArgs...), unsigned grid, unsigned block, size_t smem, cudaStream_t s,
                                    bool pdl, bool cooperative, Args... args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(grid, 1, 1);
    cfg.blockDim = dim3(block, 1, 1);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = s;
    cudaLaunchAttribute attr[2];
    int na = 0;
    if (pdl) {
        attr[na].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        attr[na].val.programmaticStreamSerializationAllowed = 1;
        ++na;
    }
    if (cooperative) {                       // grid-wide barrier inside the kernel: all CTAs co-resident
        attr[na].id = cudaLaunchAttributeCooperative;
        attr[na].val.cooperative = 1;
        ++na;
    }
    cfg.attrs = attr;
    cfg.numAttrs = na;
    return cudaLaunchKernelEx(&cfg, kernel, args...);
}
template <typename... KArgs, typename... Args>
inline cudaError_t launch_kernel(void (*kernel)(KArgs...), unsigned grid, unsigned block, size_t smem, cudaStream_t s,
                                 bool pdl, Args... args) {
    return launch_kernel_ex(kernel, grid, block, smem, s, pdl, false, args...);
}
#endif

#ifdef __CUDACC__
// ---------------------------------------------------------------------------------------------
// mbarrier / bulk-copy primitives (PTX ISA: mbarrier, cp.async.bulk)
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t *b, int cnt) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(b)), "r"(cnt));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *b, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(b)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t *b) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(b)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *b, uint32_t parity) {
    asm volatile(
        "{\n\t.reg .pred p;\n\tWAIT_%=:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra DONE_%=;\n\tbra WAIT_%=;\n\tDONE_%=:\n\t}" ::"r"(smem_u32(b)), "r"(parity) : "memory");
}
// the same wait for a warp that may have to wait LONG for another warp of its own CTA: poll, and sleep in between,
// so that the waiting warps do not take the issue slots the warp they wait for needs
__device__ __forceinline__ void mbar_wait_backoff(uint64_t *b, uint32_t parity) {
    for (;;) {
        uint32_t ok;
        asm volatile(
            "{\n\t.reg .pred p;\n\t"
            "mbarrier.test_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
            "selp.u32 %0, 1, 0, p;\n\t}" : "=r"(ok) : "r"(smem_u32(b)), "r"(parity) : "memory");
        if (ok) break;
        __nanosleep(100);
    }
}
__device__ __forceinline__ uint64_t policy_evict_first() {
    uint64_t pol;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
    return pol;
}
__device__ __forceinline__ void bulk_g2s(void *dst, const void *src, uint32_t bytes, uint64_t *bar, uint64_t pol) {
    asm volatile(
        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;"
        ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)), "l"(pol) : "memory");
}
#endif

// ---------------------------------------------------------------------------------------------
// Device helpers
// ---------------------------------------------------------------------------------------------
#ifdef __CUDACC__
// largest t in [0,T) with prefix[t] <= x  (prefix is non-decreasing, prefix[0] = 0, x < prefix[T])
template <typename I>
__device__ __forceinline__ int upper_tensor(const I *__restrict__ prefix, int T, I x) {
    int lo = 0, hi = T;                    // invariant: prefix[lo] <= x < prefix[hi]
    while (hi - lo > 1) {
        int mid = (lo + hi) >> 1;
        if (__ldg(prefix + mid) <= x) lo = mid; else hi = mid;
    }
    return lo;
}

// ---- exact accumulators (see kAccWords above) -------------------------------------------------
// acc += v for a finite v > 0 that is a multiple of 2^base: the 53-bit mantissa is cut at the 32-bit window
// boundaries and every piece is added with a 64-bit integer atomic (no return value: RED)
__device__ __forceinline__ void acc_add(unsigned long long *w, int nwords, int base, double v) {
    const long long b = __double_as_longlong(v);
    const int e = (int)((b >> 52) & 0x7ff);
    if (e == 0 || e == 0x7ff) return;                    // 0 / denormal double / non-finite: not a partial we produce
    unsigned long long m = ((unsigned long long)b & 0xfffffffffffffull) | (1ull << 52);
    int p = e - 1075 - base;                             // position of the mantissa's bit 0 in the accumulator
    if (p < 0) { m >>= -p; p = 0; }                      // (the bits shifted out are zero: v is a multiple of 2^base)
    const int k = p >> 5, s = p & 31;
    const unsigned long long lo = m << s;
    const unsigned long long hi = s ? (m >> (64 - s)) : 0ull;
    const unsigned long long p0 = lo & 0xffffffffull, p1 = lo >> 32;
    if (p0 && k < nwords) atomicAdd(w + k, p0);
    if (p1 && k + 1 < nwords) atomicAdd(w + k + 1, p1);
    if (hi && k + 2 < nwords) atomicAdd(w + k + 2, hi);
}
// the exact total of `nwords` accumulator words rounded once (to nearest even) to FP64
static __device__ __noinline__ double acc_round(const unsigned long long *w, int nwords, int base) {
    unsigned long long d[20];
    unsigned long long carry = 0ull;
    int top = -1;
    for (int k = 0; k < nwords; ++k) {
        const unsigned long long t = w[k] + carry;
        d[k] = t & 0xffffffffull;
        carry = t >> 32;
        if (d[k]) top = k;
    }
    if (top < 0) return 0.0;
    const unsigned long long hi64 = (d[top] << 32) | (top >= 1 ? d[top - 1] : 0ull);
    const unsigned long long lo32 = top >= 2 ? d[top - 2] : 0ull;
    bool sticky = false;
    for (int k = 0; k < top - 2; ++k) sticky |= d[k] != 0ull;
    const int lz = __clzll((long long)hi64);             // 0..31: d[top] != 0
    unsigned long long mant = lz ? ((hi64 << lz) | (lo32 >> (32 - lz))) : hi64;
    if (sticky || ((lo32 << lz) & 0xffffffffull)) mant |= 1ull;   // below the rounding position of a 64 -> 53 bit conversion
    return scalbn(__ull2double_rn(mant), base + 32 * top + 31 - lz - 63);
}

// The same rounding done by a whole (converged) warp on one accumulator slot, lane k holding word k: `digit` is
// the lane's 32-bit digit after carry normalisation (warp_acc_digits), the number occupies lanes [l0, l0 + nwords).
__device__ __forceinline__ void warp_acc_digits(unsigned long long v, int lane, uint32_t &digit) {
    unsigned long long lo = v & 0xffffffffull, hi = v >> 32;
    if (lane >= kAccNan) { lo = 0ull; hi = 0ull; }
    for (;;) {                                           // deferred carries ripple up (two numbers: no carry into lanes 0 / kAccSq)
        unsigned long long c = __shfl_up_sync(0xffffffffu, hi, 1);
        if (lane == kAccAbs || lane == kAccSq) c = 0ull;
        const unsigned long long s = lo + c;
        lo = s & 0xffffffffull;
        hi = s >> 32;
        if (!__any_sync(0xffffffffu, hi != 0ull)) break;
    }
    digit = (uint32_t)lo;
}
__device__ __forceinline__ double warp_acc_round(uint32_t digit, unsigned nz /*ballot(digit != 0)*/, int l0, int nwords, int base) {
    const unsigned m = (nz >> l0) & ((1u << nwords) - 1u);
    const int top = m ? 31 - __clz(m) : 0;
    const unsigned long long d0 = __shfl_sync(0xffffffffu, digit, l0 + top);
    const unsigned long long d1 = __shfl_sync(0xffffffffu, digit, l0 + max(top - 1, 0));
    const unsigned long long d2 = __shfl_sync(0xffffffffu, digit, l0 + max(top - 2, 0));
    if (m == 0u) return 0.0;
    const unsigned long long hi64 = (d0 << 32) | (top >= 1 ? d1 : 0ull);
    const unsigned long long lo32 = top >= 2 ? d2 : 0ull;
    const bool sticky = top >= 3 && (m & ((1u << (top - 2)) - 1u)) != 0u;
    const int lz = __clzll((long long)hi64);
    unsigned long long mant = lz ? ((hi64 << lz) | (lo32 >> (32 - lz))) : hi64;
    if (sticky || ((lo32 << lz) & 0xffffffffull)) mant |= 1ull;
    return scalbn(__ull2double_rn(mant), base + 32 * top + 31 - lz - 63);
}

// S_t = (float)( sum_w (double)(float)(A[w][t]/len_t) / W )   — PAPER L211 "mean-absolute scale",
// combined over workers by a fixed-order FP64 mean (readings #7, #8).
__device__ __forceinline__ float tensor_scale(const double *__restrict__ abs_sum, int W, int T, int t,
                                              int64_t len_t) {
    double s = 0.0;
    const double dl = (double)len_t;
    for (int w = 0; w < W; ++w) {
        float swt = (float)(__ldcg(abs_sum + (size_t)w * T + t) / dl);
        s += (double)swt;
    }
    return (float)(s / (double)W);
}
// The same value computed by a whole (converged) warp: the W loads of a round of 32 workers are in
// flight together (one L2 round trip per 32 workers instead of one per worker) and the FP64 adds
// run in the same fixed worker order through a shuffle chain, so the result is bit-identical.
__device__ __forceinline__ float warp_tensor_scale(const double *__restrict__ abs_sum, int W, int T, int t,
                                                   int64_t len_t, int lane) {
    double s = 0.0;
    const double dl = (double)len_t;
    for (int w0 = 0; w0 < W; w0 += 32) {
        const int w = w0 + lane;
        const float swt = (w < W) ? (float)(__ldcg(abs_sum + (size_t)w * T + t) / dl) : 0.f;
        const int cnt = min(32, W - w0);
        for (int j = 0; j < cnt; ++j) s += (double)__shfl_sync(0xffffffffu, swt, j);
    }
    return (float)(s / (double)W);
}
#endif

}  // namespace nf
