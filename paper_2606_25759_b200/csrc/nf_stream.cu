// nf_stream.cu — the stand-alone streaming calls: steps a2 (pack), a4a (FP32 route) and a4b (health),
// each one read of its input. PAPER §5.2, §3.3; SURVEY §8(a). (The fused path, which does
// all of them and the count/vote/decode from ONE read of the W x n gradients, is nf_fused.cu.)
//
// HBM-bound elementwise streaming (no contraction -> no tensor cores). Design for sm_100a:
//  * persistent grid (multiple of the SM count), CTAs walk tiles of ONE tensor (tensor-relative
//    index space), so packed bit j of word k is lane-aligned for any tensor offset;
//  * each thread owns 4 consecutive elements per row and loads them from up to 8 workers with
//    128-bit streaming loads (16 independent 16-byte requests in flight per thread);
//  * sign bits are built as one 4-bit nibble per worker in a single register (8 workers x 4 bits);
//    per-position counts are popcounts of that register under a 0x11111111 mask, and the packed
//    32-bit plane words come from an 8x8 nibble transpose across 8 lanes (3 shuffles);
//  * per-(worker,tensor) abs-sum / sum-of-squares run in FP32 over 8 elements, then FP64 per
//    thread, one fixed-shape block reduce-scatter per tensor change, and the block's total goes EXACTLY
//    into the plan's wide fixed-point accumulators (integer atomics, nf_internal.cuh): the result does
//    not depend on the order in which the CTAs arrive; finalize_kernel rounds each total to FP64 once.
#include <float.h>
#include "nf_internal.cuh"

namespace nf {

__device__ __forceinline__ float4 ld_stream4(const float *p) {
    return __ldcs(reinterpret_cast<const float4 *>(p));
}

// Load 4 consecutive floats of which the first `valid` exist; missing ones read as +0.
__device__ __forceinline__ float4 load4(const float *p, int valid, bool aligned) {
    if (valid == 4 && aligned) return ld_stream4(p);
    float4 r = make_float4(0.f, 0.f, 0.f, 0.f);
    if (valid > 0) r.x = __ldcs(p);
    if (valid > 1) r.y = __ldcs(p + 1);
    if (valid > 2) r.z = __ldcs(p + 2);
    if (valid > 3) r.w = __ldcs(p + 3);
    return r;
}

// 8x8 transpose of 4-bit elements held one row per lane across each aligned group of 8 lanes:
// in : lane q holds nibble u = M[q][u];   out: lane q holds nibble q' = M[q'][q].
// Three butterfly stages; the 16-bit and 8-bit stages are single byte-permutes (PRMT) with a
// per-lane selector, the 4-bit stage is a rotate + bit-select.
struct TransposeCtl { uint32_t sel4, sel2, rot1, mask1; };
__device__ __forceinline__ TransposeCtl make_transpose_ctl(int lane) {
    TransposeCtl c;
    c.sel4 = (lane & 4) ? 0x3276u : 0x5410u;     // [t2 t3 v2 v3] : [v0 v1 t0 t1]
    c.sel2 = (lane & 2) ? 0x3715u : 0x6240u;     // [t1 v1 t3 v3] : [v0 t0 v2 t2]
    c.rot1 = (lane & 1) ? 28u : 4u;              // t >> 4 : t << 4 (as a rotate)
    c.mask1 = (lane & 1) ? 0xf0f0f0f0u : 0x0f0f0f0fu;
    return c;
}
__device__ __forceinline__ uint32_t nibble_transpose8(uint32_t v, const TransposeCtl &c) {
    uint32_t t = __shfl_xor_sync(0xffffffffu, v, 4);
    v = __byte_perm(v, t, c.sel4);
    t = __shfl_xor_sync(0xffffffffu, v, 2);
    v = __byte_perm(v, t, c.sel2);
    t = __shfl_xor_sync(0xffffffffu, v, 1);
    t = __funnelshift_l(t, t, c.rot1);
    return (v & c.mask1) | (t & ~c.mask1);
}

// Warp reduce-scatter of 16 doubles: on return v[0] of lane l holds the warp total of value
// idx(l) = 8*bit4 + 4*bit3 + 2*bit2 + bit1 (lanes l and l^1 hold the same value). Fixed order.
__device__ __forceinline__ void warp_reduce_scatter16(double (&v)[16], int lane) {
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        const bool hi = lane & 16;
        double send = hi ? v[i] : v[i + 8], keep = hi ? v[i + 8] : v[i];
        v[i] = keep + __shfl_xor_sync(0xffffffffu, send, 16);
    }
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const bool hi = lane & 8;
        double send = hi ? v[i] : v[i + 4], keep = hi ? v[i + 4] : v[i];
        v[i] = keep + __shfl_xor_sync(0xffffffffu, send, 8);
    }
#pragma unroll
    for (int i = 0; i < 2; ++i) {
        const bool hi = lane & 4;
        double send = hi ? v[i] : v[i + 2], keep = hi ? v[i + 2] : v[i];
        v[i] = keep + __shfl_xor_sync(0xffffffffu, send, 4);
    }
    {
        const bool hi = lane & 2;
        double send = hi ? v[0] : v[1], keep = hi ? v[1] : v[0];
        v[0] = keep + __shfl_xor_sync(0xffffffffu, send, 2);
    }
    v[0] += __shfl_xor_sync(0xffffffffu, v[0], 1);
}

struct FlushCtx {
    double (*s_red)[16];
    unsigned int *s_nan;
    unsigned int *s_inf;
    unsigned long long *acc;    // the plan's exact accumulators, [W*T][kAccWords]
};

// Block-reduce the per-thread FP64 partials of one worker group (fixed shape: with the static tile striding of
// this kernel the value is a function of the data and the grid size only) and add the block's totals exactly
// to the per-(worker,tensor) accumulators; NaN / Inf are tallied, never added. CTA-uniform call.
template <int FLAGS>
__device__ __forceinline__ void flush_stats(const StreamParams &p, const FlushCtx &c, double (&a)[8],
                                            double (&q)[8], int w0, int nw, int t, bool isL) {
    constexpr bool PACK = FLAGS & kFPack, HEALTH = FLAGS & kFHealth;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    double v[16];
#pragma unroll
    for (int i = 0; i < 8; ++i) { v[i] = a[i]; v[i + 8] = q[i]; a[i] = 0.0; q[i] = 0.0; }
    warp_reduce_scatter16(v, lane);
    const int idx = ((lane >> 4) & 1) * 8 + ((lane >> 3) & 1) * 4 + ((lane >> 2) & 1) * 2 + ((lane >> 1) & 1);
    if ((lane & 1) == 0) c.s_red[warp][idx] = v[0];
    __syncthreads();
    if (threadIdx.x < 16) {
        const int j = threadIdx.x, w = j & 7;
        double tot = 0.0;
#pragma unroll
        for (int k = 0; k < kThreads / 32; ++k) tot += c.s_red[k][j];
        if (w < nw) {
            unsigned long long *slot = c.acc + ((size_t)(w0 + w) * p.T + t) * kAccWords;
            if (j < 8) {
                if (PACK && isL) acc_add(slot + kAccAbs, kAccAbsWords, kAccAbsBase, tot);
            } else {
                if (HEALTH) acc_add(slot + kAccSq, kAccSqWords, kAccSqBase, tot);
            }
        }
    } else if (threadIdx.x >= 32 && threadIdx.x < 40) {
        const int w = threadIdx.x - 32;
        const unsigned int cn = c.s_nan[w], ci = c.s_inf[w];
        if (w < nw && (HEALTH || isL)) {
            unsigned long long *slot = c.acc + ((size_t)(w0 + w) * p.T + t) * kAccWords;
            if (cn) atomicAdd(slot + kAccNan, (unsigned long long)cn);
            if (ci) atomicAdd(slot + kAccInf, (unsigned long long)ci);
        }
        c.s_nan[w] = 0u;
        c.s_inf[w] = 0u;
    }
    __syncthreads();
}

// pos/neg indicator bits: one compare + one predicated OR per element and plane
__device__ __forceinline__ void or_if_gt(uint32_t &r, float x, float t, uint32_t bit) {
    asm("{\n\t.reg .pred p;\n\tsetp.gt.f32 p, %1, %2;\n\t@p or.b32 %0, %0, %3;\n\t}" : "+r"(r) : "f"(x), "f"(t), "r"(bit));
}
__device__ __forceinline__ void or_if_lt(uint32_t &r, float x, float t, uint32_t bit) {
    asm("{\n\t.reg .pred p;\n\tsetp.lt.f32 p, %1, %2;\n\t@p or.b32 %0, %0, %3;\n\t}" : "+r"(r) : "f"(x), "f"(t), "r"(bit));
}

template <bool B> struct BoolTag { static constexpr bool value = B; };
template <int I> struct IntTag { static constexpr int value = I; };

// Element owned by (warp, lane) in row u of a tile: each warp covers 256 consecutive elements per
// tile (two rows of 128), so its packed words of one worker are 8 consecutive words = one 32-byte
// sector, its direction bytes one sector per row, and every load/store instruction is 512 B wide.
__device__ __forceinline__ int tile_elem(int warp, int lane, int u) { return warp * (kRows * 128) + u * 128 + lane * 4; }

template <int FLAGS>
__global__ void __launch_bounds__(kThreads, 2) stream_kernel(const StreamParams p) {
    constexpr bool PACK = FLAGS & kFPack, FP32 = FLAGS & kFFp32, HEALTH = FLAGS & kFHealth;
    constexpr bool STATS = PACK || HEALTH;
    __shared__ double s_red[kThreads / 32][16];
    __shared__ unsigned int s_nan[8], s_inf[8];
    pdl_launch_dependents();
    pdl_wait();
    const PlanView pv = plan_view(p.plan, p.T);
    if (pv.hdr->magic != kPlanMagic || pv.hdr->status != NF_OK) return;
    if (STATS && (int64_t)p.W * p.T > pv.hdr->acc_slots) return;      // plan too small: finalize_kernel reports it
    if (PACK && p.P && pv.hdr->Wd > p.plane_stride) return;           // plane rows too short: likewise
    const int n_tiles = pv.hdr->n_tiles;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid < 8) { s_nan[tid] = 0u; s_inf[tid] = 0u; }
    __syncthreads();
    const FlushCtx fc{s_red, s_nan, s_inf, pv.acc};
    const TransposeCtl tctl = make_transpose_ctl(lane);

    const int W = p.W;
    const bool multi = W > kGroup;           // more than one register group of workers
    const bool ternary = p.ternary != 0;
    double a[8], q[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) { a[i] = 0.0; q[i] = 0.0; }
    int acc_t = -1;                          // tensor the accumulators belong to (single-group mode)
    bool acc_isL = false;

    // cached properties of the current tensor
    int t = -1, tile_b = 0, tile_e = 0;
    int64_t off_t = 0, len_t = 0, woff_t = 0;
    bool isL = false, aligned = false;
    float tau = 0.f, ntau = -0.f;

    for (int tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
        if (tile >= tile_e) {
            t = upper_tensor<int32_t>(pv.tile_prefix, p.T, tile);
            tile_b = __ldg(pv.tile_prefix + t);
            tile_e = __ldg(pv.tile_prefix + t + 1);
            off_t = __ldg(p.off + t);
            len_t = __ldg(p.len + t);
            isL = p.route ? (__ldg(p.route + t) == NF_ROUTE_L) : false;
            woff_t = (isL && p.woff) ? __ldg(p.woff + t) : 0;
            tau = (p.tau && isL) ? __ldg(p.tau + t) : 0.f;
            ntau = -tau;
            aligned = (((off_t | p.worker_stride) & 3) == 0);
        }
        const bool do_tile = HEALTH || (isL ? PACK : FP32);
        if (!do_tile) continue;
        if (STATS && !multi && acc_t != t) {
            if (acc_t >= 0) flush_stats<FLAGS>(p, fc, a, q, 0, W, acc_t, acc_isL);
            acc_t = t;
            acc_isL = isL;
        }
        const int64_t tile_base = (int64_t)(tile - tile_b) * kTile;   // tensor-relative
        const bool full_tile = aligned && (len_t - tile_base >= kTile);
        int64_t irel[kRows];
        int valid[kRows];
#pragma unroll
        for (int u = 0; u < kRows; ++u) {
            irel[u] = tile_base + tile_elem(warp, lane, u);
            const int64_t rem = len_t - irel[u];
            valid[u] = rem >= 4 ? 4 : (rem > 0 ? (int)rem : 0);
        }
        uint32_t posR[kRows], negR[kRows];
        float4 acc[kRows];                   // FP32-route running sums
#pragma unroll
        for (int u = 0; u < kRows; ++u) acc[u] = make_float4(0.f, 0.f, 0.f, 0.f);

        for (int w0 = 0; w0 < W; w0 += kGroup) {
            const int nw = min(kGroup, W - w0);
            const float *gb = p.g + (size_t)w0 * p.worker_stride + off_t;
#pragma unroll
            for (int u = 0; u < kRows; ++u) { posR[u] = 0u; negR[u] = 0u; }

            auto body = [&](auto full_tag, auto kind_tag) {
                constexpr bool FULL = decltype(full_tag)::value;   // 8 workers, whole aligned tile
                constexpr int KIND = decltype(kind_tag)::value;    // 0: non-L tile, 1: L G-Binary, 2: L G-Ternary
                float4 x[kRows][kGroup];
#pragma unroll
                for (int u = 0; u < kRows; ++u)
#pragma unroll
                    for (int w = 0; w < kGroup; ++w) {
                        const float *src = gb + (size_t)w * p.worker_stride + irel[u];
                        if (FULL) x[u][w] = ld_stream4(src);
                        else x[u][w] = (w < nw) ? load4(src, valid[u], aligned) : make_float4(0.f, 0.f, 0.f, 0.f);
                    }
                if (FULL) {
                    // pull the unit this CTA visits next into L2 while this one is being computed:
                    // 8 workers x 1 KB per warp = 64 lines, two per lane
                    const float *nb = nullptr;
                    if (w0 + 2 * kGroup <= W) nb = gb + (size_t)kGroup * p.worker_stride + tile_base;
                    else if (w0 + kGroup >= W && tile + (int)gridDim.x < tile_e &&
                             len_t - (tile_base + (int64_t)gridDim.x * kTile) >= kTile)
                        nb = p.g + off_t + tile_base + (int64_t)gridDim.x * kTile;
                    if (nb) {
                        const float *l = nb + (size_t)(lane >> 2) * p.worker_stride + warp * (kRows * 128) + (lane & 3) * 32;
                        asm volatile("prefetch.global.L2 [%0];" ::"l"(l));
                        asm volatile("prefetch.global.L2 [%0];" ::"l"(l + 128));
                    }
                }
                uint32_t badmask = 0u;
#pragma unroll
                for (int w = 0; w < kGroup; ++w) {
                    if (!FULL && w >= nw) continue;
                    if (STATS) {
                        // FP32 over this thread's 8 elements of worker w, then FP64
                        float af = 0.f, qf = 0.f;
#pragma unroll
                        for (int u = 0; u < kRows; ++u) {
                            const float4 v = x[u][w];
                            af += (fabsf(v.x) + fabsf(v.y)) + (fabsf(v.z) + fabsf(v.w));
                            if (HEALTH) {
                                qf = fmaf(v.x, v.x, qf); qf = fmaf(v.y, v.y, qf);
                                qf = fmaf(v.z, v.z, qf); qf = fmaf(v.w, v.w, qf);
                            }
                        }
                        // fast path: everything finite and the FP32 squares did not underflow
                        const bool ok = HEALTH ? (((qf >= 1e-30f) && (qf < FLT_MAX)) || af == 0.f)
                                               : (af < FLT_MAX);
                        a[w] += (double)(ok ? af : 0.f);
                        if (HEALTH) q[w] += (double)(ok ? qf : 0.f);
                        badmask |= ok ? 0u : (1u << w);
                    }
                    if (KIND != 0) {
                        if (PACK) {
#pragma unroll
                            for (int u = 0; u < kRows; ++u) {
                                const float4 v = x[u][w];
                                or_if_gt(posR[u], v.x, tau, 1u << (4 * w));
                                or_if_gt(posR[u], v.y, tau, 2u << (4 * w));
                                or_if_gt(posR[u], v.z, tau, 4u << (4 * w));
                                or_if_gt(posR[u], v.w, tau, 8u << (4 * w));
                                if (KIND == 2) {
                                    or_if_lt(negR[u], v.x, ntau, 1u << (4 * w));
                                    or_if_lt(negR[u], v.y, ntau, 2u << (4 * w));
                                    or_if_lt(negR[u], v.z, ntau, 4u << (4 * w));
                                    or_if_lt(negR[u], v.w, ntau, 8u << (4 * w));
                                }
                            }
                        }
                    } else if (FP32) {
                        // fixed worker order, plain FP32 adds
#pragma unroll
                        for (int u = 0; u < kRows; ++u) {
                            const float4 v = x[u][w];
                            if (w == 0 && w0 == 0) acc[u] = v;
                            else {
                                acc[u].x = __fadd_rn(acc[u].x, v.x); acc[u].y = __fadd_rn(acc[u].y, v.y);
                                acc[u].z = __fadd_rn(acc[u].z, v.z); acc[u].w = __fadd_rn(acc[u].w, v.w);
                            }
                        }
                    }
                }
                if (STATS && badmask) {
                    // rare: NaN / Inf / FP32 over- or underflow in this thread's elements -> FP64, exact tallies
#pragma unroll
                    for (int w = 0; w < kGroup; ++w) {
                        if (!((badmask >> w) & 1u)) continue;
#pragma unroll
                        for (int u = 0; u < kRows; ++u) {
                            const float e4[4] = {x[u][w].x, x[u][w].y, x[u][w].z, x[u][w].w};
#pragma unroll
                            for (int j = 0; j < 4; ++j) {
                                const float v = e4[j];
                                if (v != v) atomicAdd(&s_nan[w], 1u);
                                else if (fabsf(v) == INFINITY) atomicAdd(&s_inf[w], 1u);
                                else {
                                    a[w] += (double)fabsf(v);
                                    if (HEALTH) q[w] += (double)v * (double)v;
                                }
                            }
                        }
                    }
                }
            };
            const int kind = isL ? (ternary ? 2 : 1) : 0;
            if (full_tile && nw == kGroup) {
                if (kind == 2) body(BoolTag<true>{}, IntTag<2>{});
                else if (kind == 1) body(BoolTag<true>{}, IntTag<1>{});
                else body(BoolTag<true>{}, IntTag<0>{});
            } else {
                if (kind == 2) body(BoolTag<false>{}, IntTag<2>{});
                else if (kind == 1) body(BoolTag<false>{}, IntTag<1>{});
                else body(BoolTag<false>{}, IntTag<0>{});
            }

            if (isL && PACK) {
                if (PACK && p.P) {
                    const int wq = lane & 7;
                    const int64_t nwords = (len_t + 31) >> 5;
#pragma unroll
                    for (int u = 0; u < kRows; ++u) {
                        const int64_t wi = (tile_base >> 5) + warp * (kRows * 4) + u * 4 + (lane >> 3);
                        const bool st = (wq < nw) && (wi < nwords);
                        const size_t o = (size_t)(w0 + wq) * p.plane_stride + woff_t + wi;
                        const uint32_t pw = nibble_transpose8(posR[u], tctl);
                        if (st) p.P[o] = pw;
                        if (ternary) {
                            const uint32_t nwd = nibble_transpose8(negR[u], tctl);
                            if (st) p.N[o] = nwd;
                        }
                    }
                }
            }
            if (multi && STATS) flush_stats<FLAGS>(p, fc, a, q, w0, nw, t, isL);
        }

        if (!isL && FP32) {
#pragma unroll
            for (int u = 0; u < kRows; ++u) {
                float *o = p.out + off_t + irel[u];
                float4 r = acc[u];
                r.x = __fmul_rn(p.alpha, r.x); r.y = __fmul_rn(p.alpha, r.y);
                r.z = __fmul_rn(p.alpha, r.z); r.w = __fmul_rn(p.alpha, r.w);
                if (valid[u] == 4 && ((off_t & 3) == 0)) {
                    __stcs(reinterpret_cast<float4 *>(o), r);
                } else {
                    if (valid[u] > 0) o[0] = r.x;
                    if (valid[u] > 1) o[1] = r.y;
                    if (valid[u] > 2) o[2] = r.z;
                    if (valid[u] > 3) o[3] = r.w;
                }
            }
        }
    }
    if (STATS && !multi && acc_t >= 0) flush_stats<FLAGS>(p, fc, a, q, 0, W, acc_t, acc_isL);
}

// ---------------------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------------------
int device_sm_count() {
    static int sms = 0;
    if (sms == 0) {
        int dev = 0;
        if (cudaGetDevice(&dev) != cudaSuccess) return 148;
        if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms <= 0)
            sms = 148;
    }
    return sms;
}

// Rounds the exact totals of every (replica, tensor) slot to FP64 once, writes the call's outputs and clears the
// slots (one thread per slot). FLAGS as in stream_kernel. A plan whose accumulator region is too small for W x T
// slots is reported by poisoning the plan (status NF_ERR_ARG), like a bad layout.
template <int FLAGS>
__global__ void __launch_bounds__(128) finalize_kernel(const StreamParams p) {
    constexpr bool PACK = FLAGS & kFPack, HEALTH = FLAGS & kFHealth;
    pdl_launch_dependents();
    pdl_wait();
    const PlanView pv = plan_view(p.plan, p.T);
    if (pv.hdr->magic != kPlanMagic || pv.hdr->status != NF_OK) return;
    const int64_t slots = (int64_t)p.W * p.T;
    if (slots > pv.hdr->acc_slots || (PACK && p.P && pv.hdr->Wd > p.plane_stride)) {
        if (blockIdx.x == 0 && threadIdx.x == 0) const_cast<PlanHeader *>(pv.hdr)->status = NF_ERR_ARG;
        return;
    }
    const int64_t o = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (o >= slots) return;
    const int t = (int)(o % p.T);
    unsigned long long wd[kAccWords];
    ulonglong2 *slot = reinterpret_cast<ulonglong2 *>(pv.acc + (size_t)o * kAccWords);
#pragma unroll
    for (int i = 0; i < kAccWords / 2; ++i) {
        const ulonglong2 v = __ldcg(slot + i);
        wd[2 * i] = v.x;
        wd[2 * i + 1] = v.y;
    }
#pragma unroll
    for (int i = 0; i < kAccWords / 2; ++i) __stcg(slot + i, make_ulonglong2(0ull, 0ull));
    const unsigned long long cn = wd[kAccNan], ci = wd[kAccInf];
    if (PACK) {
        double A = 0.0;
        if (p.route[t] == NF_ROUTE_L) {
            A = acc_round(wd + kAccAbs, kAccAbsWords, kAccAbsBase);
            if (cn) A = __longlong_as_double(0x7ff8000000000000ll);          // IEEE: NaN term -> NaN, Inf term -> +Inf
            else if (ci) A = __longlong_as_double(0x7ff0000000000000ll);
        }
        p.abs_sum[o] = A;
    }
    if (HEALTH) {
        p.sumsq[o] = acc_round(wd + kAccSq, kAccSqWords, kAccSqBase);
        p.nan_cnt[o] = cn;
        p.inf_cnt[o] = ci;
    }
}

template <int FLAGS>
static cudaError_t launch_stream_t(const StreamParams &p, int64_t n, cudaStream_t s) {
    static int per_sm = 0;
    if (per_sm == 0) {
        if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, stream_kernel<FLAGS>, kThreads, 0) !=
                cudaSuccess || per_sm <= 0)
            per_sm = 1;
    }
    // upper bound of the tile count known on the host: every tensor adds at most one ragged tile
    const int64_t max_tiles = n / kTile + p.T;
    if (max_tiles <= 0) return cudaSuccess;
    int64_t grid = (int64_t)device_sm_count() * per_sm;     // persistent: a multiple of the SM count
    if (grid > max_tiles) grid = max_tiles;
    cudaError_t e = launch_kernel(stream_kernel<FLAGS>, (unsigned)grid, kThreads, 0, s, true, p);
    if (e != cudaSuccess) return e;
    if (FLAGS & (kFPack | kFHealth)) {
        const int64_t slots = (int64_t)p.W * p.T;
        e = launch_kernel(finalize_kernel<FLAGS>, (unsigned)((slots + 127) / 128), 128, 0, s, true, p);
        if (e != cudaSuccess) return e;
    }
    return cudaGetLastError();
}

cudaError_t launch_stream(int flags, const StreamParams &p, int64_t n, cudaStream_t s) {
    switch (flags) {
        case kFPack: return launch_stream_t<kFPack>(p, n, s);
        case kFFp32: return launch_stream_t<kFFp32>(p, n, s);
        case kFHealth: return launch_stream_t<kFHealth>(p, n, s);
        default: return cudaErrorInvalidValue;
    }
}

}  // namespace nf
