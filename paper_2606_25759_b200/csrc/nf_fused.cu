// nf_fused.cu — pass A of the fused path (nf_aggregate_bucket): route-aware pack + sign count +
// majority vote + FP32-route sum + abs-sums + health statistics from ONE read of the W x n
// gradients. PAPER §5.2, §3.3; SURVEY §8(a) a2/a3/a4a/a4b, §8(d) "fused floor".
//
// Blackwell design (HBM-bound streaming, no contraction -> no tensor cores):
//  * one persistent CTA per SM: 16 consumer warps + 1 producer warp (+ decode warps, see below);
//  * the producer's elected lane streams tiles (2048 elements x 8 workers = 64 KB) from HBM into a
//    shared-memory ring with 1-D bulk async copies (cp.async.bulk, the TMA engine) that complete on
//    an mbarrier, with an L2 evict-first policy (the gradients are read exactly once); the
//    bytes in flight no longer depend on registers or occupancy;
//  * consumer warps wait on the stage's "full" mbarrier, pull their 8 float4 (conflict-free
//    LDS.128), release the stage at once ("empty" mbarrier) and only then compute;
//  * per thread: 4 consecutive elements of up to 8 workers -> one 4-bit nibble per worker in one
//    register per plane; counts are popcounts under a 0x11111111 mask; packed plane words come
//    from an 8x8 nibble transpose across 8 lanes;
//  * abs-sum / sum of squares: FP32 partials over kKTiles tiles (<= 16 elements, pairwise inside a
//    float4), then FP64 per thread; a failed range check (NaN, Inf, FP32 over/underflow) sends the
//    thread to an exact FP64 re-read of just those elements.
// Tiles whose rows cannot be bulk-copied (tensor rows not 16-byte aligned, or a tail that would
// read past the bucket) take a generic predicated path straight from global memory.
#include <float.h>
#include "nf_internal.cuh"

namespace nf {

constexpr int kCW = 16;                          // consumer warps
constexpr int kCThreads = kCW * 32;              // 512 threads x 4 elements = one tile
constexpr int kFThreads = kCThreads + 64;         // + producer warp + tail warp
constexpr int kStageFloats = kGroup * kTile;     // 8 workers x 2048 elements
constexpr int kStageBytes = kStageFloats * 4;    // 64 KB
constexpr int kKTiles = 4;                       // tiles of FP32 partial accumulation
constexpr int kMaxStages = 4;
constexpr int kStages = 3;                       // ring depth: 3 x 64 KB
static_assert(kTile == kCThreads * 4, "one float4 per consumer thread per worker and tile");

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
// barrier among the consumer warps only (the producer / decode warps never join it)
__device__ __forceinline__ void consumer_sync() { asm volatile("bar.sync 1, %0;" ::"n"(kCThreads) : "memory"); }

// ---------------------------------------------------------------------------------------------
// small helpers shared with the LDG kernels (re-stated here: this TU is self-contained)
// ---------------------------------------------------------------------------------------------
struct TCtl { uint32_t sel4, sel2, rot1, mask1; };
__device__ __forceinline__ TCtl make_tctl(int lane) {
    TCtl c;
    c.sel4 = (lane & 4) ? 0x3276u : 0x5410u;
    c.sel2 = (lane & 2) ? 0x3715u : 0x6240u;
    c.rot1 = (lane & 1) ? 28u : 4u;
    c.mask1 = (lane & 1) ? 0xf0f0f0f0u : 0x0f0f0f0fu;
    return c;
}
// 8x8 transpose of 4-bit elements across each aligned group of 8 lanes:
// in: lane q holds nibble u = M[q][u]; out: lane q holds nibble q' = M[q'][q].
__device__ __forceinline__ uint32_t nib_transpose8(uint32_t v, const TCtl &c) {
    uint32_t t = __shfl_xor_sync(0xffffffffu, v, 4);
    v = __byte_perm(v, t, c.sel4);
    t = __shfl_xor_sync(0xffffffffu, v, 2);
    v = __byte_perm(v, t, c.sel2);
    t = __shfl_xor_sync(0xffffffffu, v, 1);
    t = __funnelshift_l(t, t, c.rot1);
    return (v & c.mask1) | (t & ~c.mask1);
}
__device__ __forceinline__ void or_gt(uint32_t &r, float x, float t, uint32_t bit) {
    asm("{\n\t.reg .pred p;\n\tsetp.gt.f32 p, %1, %2;\n\t@p or.b32 %0, %0, %3;\n\t}" : "+r"(r) : "f"(x), "f"(t), "r"(bit));
}
__device__ __forceinline__ void or_lt(uint32_t &r, float x, float t, uint32_t bit) {
    asm("{\n\t.reg .pred p;\n\tsetp.lt.f32 p, %1, %2;\n\t@p or.b32 %0, %0, %3;\n\t}" : "+r"(r) : "f"(x), "f"(t), "r"(bit));
}

// index of the value a lane holds after reduce_scatter16: 8*bit4 + 4*bit3 + 2*bit2 + bit1
__device__ __forceinline__ int rs16_index(int lane) {
    return ((lane >> 4) & 1) * 8 + ((lane >> 3) & 1) * 4 + ((lane >> 2) & 1) * 2 + ((lane >> 1) & 1);
}
template <typename F>
__device__ __forceinline__ F reduce_scatter16(F (&v)[16], int lane) {
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        const bool hi = lane & 16;
        F send = hi ? v[i] : v[i + 8], keep = hi ? v[i + 8] : v[i];
        v[i] = keep + __shfl_xor_sync(0xffffffffu, send, 16);
    }
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const bool hi = lane & 8;
        F send = hi ? v[i] : v[i + 4], keep = hi ? v[i + 4] : v[i];
        v[i] = keep + __shfl_xor_sync(0xffffffffu, send, 8);
    }
#pragma unroll
    for (int i = 0; i < 2; ++i) {
        const bool hi = lane & 4;
        F send = hi ? v[i] : v[i + 2], keep = hi ? v[i + 2] : v[i];
        v[i] = keep + __shfl_xor_sync(0xffffffffu, send, 4);
    }
    {
        const bool hi = lane & 2;
        F send = hi ? v[0] : v[1], keep = hi ? v[1] : v[0];
        v[0] = keep + __shfl_xor_sync(0xffffffffu, send, 2);
    }
    return v[0] + __shfl_xor_sync(0xffffffffu, v[0], 1);
}

// ---------------------------------------------------------------------------------------------
// shared-memory carve-up (dynamic). Everything the hot loop touches sits at a compile-time offset:
//   [0, 64)      mbarriers full[4], empty[4]
//   [64, 2112)   NaN / Inf tallies, 256 workers each
//   [4096, ...)  ring [stages][8][kTile] floats
//   after ring   per-warp FP64 totals {abs, sq} per worker: [kCW][2*W] doubles
// ---------------------------------------------------------------------------------------------
constexpr int kSmemHdr = 4096;
struct FusedSmem {
    float *ring;
    uint64_t *full, *empty;
    unsigned int *nan, *inf;
    double *wacc;
};
__host__ __device__ inline size_t fused_smem_bytes(int stages, int W) {
    return (size_t)kSmemHdr + (size_t)stages * kStageBytes + sizeof(double) * kCW * 2 * (size_t)W;
}
__device__ __forceinline__ FusedSmem carve(unsigned char *base, int stages) {
    FusedSmem s;
    s.full = (uint64_t *)base;
    s.empty = s.full + kMaxStages;
    s.nan = (unsigned int *)(base + 64);
    s.inf = s.nan + 256;
    s.ring = (float *)(base + kSmemHdr);
    s.wacc = (double *)(base + kSmemHdr + (size_t)stages * kStageBytes);
    return s;
}

// properties of the tensor a warp role is currently walking
struct TensorCur {
    int t, tile_b, tile_e;
    int64_t off, len, woff;
    bool isL, aligned;
    float tau;
};
__device__ __forceinline__ void tensor_lookup(const StreamParams &p, const PlanView &pv, int tile, TensorCur &c) {
    const int t = upper_tensor<int32_t>(pv.tile_prefix, p.T, tile);
    c.t = t;
    c.tile_b = __ldg(pv.tile_prefix + t);
    c.tile_e = __ldg(pv.tile_prefix + t + 1);
    c.off = __ldg(p.off + t);
    c.len = __ldg(p.len + t);
    c.isL = __ldg(p.route + t) == NF_ROUTE_L;
    c.woff = c.isL ? __ldg(p.woff + t) : 0;
    c.tau = (p.tau && c.isL) ? __ldg(p.tau + t) : 0.f;
    c.aligned = (((c.off | p.worker_stride) & 3) == 0);
}
// Exact FP64 re-read of one thread's elements of worker `wg` over the last `cnt` bulk tiles of the
// current tensor (rare: NaN / Inf / FP32 range trouble in the FP32 partials). Returns
// {sum |x|, sum of x^2 over finite x}; NaN / Inf are tallied in shared memory slot `slot`.
template <bool HEALTH>
__device__ __noinline__ double2 exact_redo(const float *__restrict__ g, int64_t worker_stride, int wg,
                                           int64_t off_t, int64_t len_t, int tile_b, int last_tile, int cnt,
                                           int tile_step, int ctid, unsigned int *s_nan, unsigned int *s_inf,
                                           int slot) {
    double da = 0.0, dq = 0.0;
    const float *row = g + (size_t)wg * worker_stride + off_t;
    for (int j = 0; j < cnt; ++j) {
        const int64_t base = (int64_t)(last_tile - j * tile_step - tile_b) * kTile + 4 * ctid;
        for (int k = 0; k < 4; ++k) {
            const int64_t i = base + k;
            if (i >= len_t) break;
            const float v = __ldg(row + i);
            da += (double)fabsf(v);
            if (HEALTH) {
                if (v != v) atomicAdd(&s_nan[slot], 1u);
                else if (fabsf(v) == INFINITY) atomicAdd(&s_inf[slot], 1u);
                else dq += (double)v * (double)v;
            }
        }
    }
    return make_double2(da, dq);
}

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int d = 16; d >= 1; d >>= 1) v += __shfl_xor_sync(0xffffffffu, v, d);
    return v;
}
__device__ __forceinline__ unsigned warp_sum(unsigned v) {
#pragma unroll
    for (int d = 16; d >= 1; d >>= 1) v += __shfl_xor_sync(0xffffffffu, v, d);
    return v;
}

// ---------------------------------------------------------------------------------------------
// fast path: a full tile of a 16-byte-aligned tensor, one worker group (W <= 8), data in the ring
// ---------------------------------------------------------------------------------------------
// L tile: sign indicators of this thread's 4 elements of every worker (nibble w of posR / negR) and
// the FP32 abs / square partials. KIND 1 = G-Binary, 2 = G-Ternary.
template <int KIND, bool HEALTH, bool FULLW>
__device__ __forceinline__ void fast_signs(const float *sb, int nw, float tau, float ntau, float (&af)[8],
                                           float (&qf)[8], uint32_t &posR, uint32_t &negR) {
#pragma unroll
    for (int w = 0; w < kGroup; ++w) {
        if (!FULLW && w >= nw) break;
        const float4 v = *reinterpret_cast<const float4 *>(sb + w * kTile);
        af[w] += (fabsf(v.x) + fabsf(v.y)) + (fabsf(v.z) + fabsf(v.w));
        if (HEALTH) {
            qf[w] = fmaf(v.x, v.x, qf[w]); qf[w] = fmaf(v.y, v.y, qf[w]);
            qf[w] = fmaf(v.z, v.z, qf[w]); qf[w] = fmaf(v.w, v.w, qf[w]);
        }
        or_gt(posR, v.x, tau, 1u << (4 * w));
        or_gt(posR, v.y, tau, 2u << (4 * w));
        or_gt(posR, v.z, tau, 4u << (4 * w));
        or_gt(posR, v.w, tau, 8u << (4 * w));
        if (KIND == 2) {
            or_lt(negR, v.x, ntau, 1u << (4 * w));
            or_lt(negR, v.y, ntau, 2u << (4 * w));
            or_lt(negR, v.z, ntau, 4u << (4 * w));
            or_lt(negR, v.w, ntau, 8u << (4 * w));
        }
    }
}
// FP32-route tile: fixed worker order, plain FP32 adds
template <bool HEALTH, bool FULLW>
__device__ __forceinline__ float4 fast_fp32(const float *sb, int nw, float (&af)[8], float (&qf)[8]) {
    float4 acc = *reinterpret_cast<const float4 *>(sb);
#pragma unroll
    for (int w = 0; w < kGroup; ++w) {
        if (!FULLW && w >= nw) break;
        const float4 v = (w == 0) ? acc : *reinterpret_cast<const float4 *>(sb + w * kTile);
        if (HEALTH) {
            af[w] += (fabsf(v.x) + fabsf(v.y)) + (fabsf(v.z) + fabsf(v.w));
            qf[w] = fmaf(v.x, v.x, qf[w]); qf[w] = fmaf(v.y, v.y, qf[w]);
            qf[w] = fmaf(v.z, v.z, qf[w]); qf[w] = fmaf(v.w, v.w, qf[w]);
        }
        if (w > 0) {
            acc.x = __fadd_rn(acc.x, v.x); acc.y = __fadd_rn(acc.y, v.y);
            acc.z = __fadd_rn(acc.z, v.z); acc.w = __fadd_rn(acc.w, v.w);
        }
    }
    return acc;
}
// majority vote of one thread's 4 positions, single worker group (readings #3, #5, #6):
// low nibble = "+" flags, high nibble = "-" flags
template <bool TERNARY>
__device__ __forceinline__ uint32_t vote4(uint32_t posR, uint32_t negR, int W, int margin) {
    uint32_t d = 0u;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        const int c_p = __popc(posR & (0x11111111u << j));
        const int c_n = TERNARY ? __popc(negR & (0x11111111u << j)) : W - c_p;
        const int D = c_p - c_n;
        if (D > margin) d |= 1u << j;
        if (D < -margin) d |= 16u << j;
    }
    return d;
}

// FP32 partials of worker group [w0, w0+nw) over the last `cnt` bulk tiles -> warp totals (FP32
// butterfly reduce-scatter) -> this warp's FP64 slots in shared memory. Range check on the warp
// totals: |x| sums finite, squares neither over- nor underflowed; otherwise the warp re-reads
// exactly those elements in FP64 (and tallies NaN / Inf).
template <bool HEALTH>
__device__ __forceinline__ void stat_flush(const StreamParams &p, const FusedSmem &sm, float (&af)[8], float (&qf)[8],
                                           int64_t off_t, int64_t len_t, int tile_b, int w0, int nw, int cnt,
                                           int last_tile, int tile_step, int ctid) {
    const int lane = ctid & 31, warp = ctid >> 5, W = p.W;
    float v16[16];
#pragma unroll
    for (int i = 0; i < 8; ++i) { v16[i] = af[i]; v16[i + 8] = qf[i]; }
    const float r = reduce_scatter16(v16, lane);
    const int idx = rs16_index(lane), wl = idx & 7, stat = idx >> 3;
    const float other = __shfl_xor_sync(0xffffffffu, r, 16);
    const float A = stat ? other : r, Q = stat ? r : other;
    const bool ok = HEALTH ? ((A <= FLT_MAX) && (((Q >= 1e-30f) && (Q <= FLT_MAX)) || A == 0.f))
                           : (A <= FLT_MAX);
    const unsigned bad = __ballot_sync(0xffffffffu, !ok && wl < nw);
    double *slot = sm.wacc + (size_t)warp * 2 * W + (size_t)w0 * 2;
    if (bad == 0u) {
        if ((lane & 1) == 0 && wl < nw) slot[wl * 2 + stat] += (double)r;
    } else {
        // rare: some worker's warp totals failed the range check. For those workers every thread
        // re-checks its own partials and only the offending threads re-read their elements exactly.
#pragma unroll
        for (int w = 0; w < kGroup; ++w) {
            if (w >= nw) break;
            const int l0 = ((w & 1) << 1) | (((w >> 1) & 1) << 2) | (((w >> 2) & 1) << 3);
            if (((bad >> l0) | (bad >> (l0 + 16))) & 1u) {
                const float a_t = af[w], q_t = qf[w];
                const bool ok_t = HEALTH ? ((a_t <= FLT_MAX) && (((q_t >= 1e-30f) && (q_t <= FLT_MAX)) || a_t == 0.f))
                                         : (a_t <= FLT_MAX);
                double2 e = make_double2((double)a_t, (double)q_t);
                if (!ok_t)
                    e = exact_redo<HEALTH>(p.g, p.worker_stride, w0 + w, off_t, len_t, tile_b, last_tile, cnt,
                                           tile_step, ctid, sm.nan, sm.inf, w0 + w);
                const double ea = warp_sum(e.x), eq = warp_sum(e.y);
                if (lane == 0) { slot[w * 2] += ea; slot[w * 2 + 1] += eq; }
            } else if ((lane & 1) == 0 && wl == w) {
                slot[w * 2 + stat] += (double)r;
            }
        }
    }
#pragma unroll
    for (int i = 0; i < 8; ++i) { af[i] = 0.f; qf[i] = 0.f; }
    __syncwarp();
}

// ---------------------------------------------------------------------------------------------
// tail warp: the LAST tile of every 16-byte-aligned tensor (the only tile that can be ragged),
// straight from global memory, one warp per tile, 128 elements per step. Runs beside the
// consumers; statistics are exact FP64 and go to the global accumulators with one warp-reduced
// atomic per worker. Same arithmetic as the fast path (oracle O2-O4b).
// ---------------------------------------------------------------------------------------------
template <bool HEALTH>
__device__ __forceinline__ void tail_tile_warp(const StreamParams &p, const TensorCur &c, int lane) {
    const int W = p.W, T = p.T;
    const bool ternary = p.ternary != 0;
    const TCtl tctl = make_tctl(lane);
    const float tau = c.tau, ntau = -c.tau;
    const int64_t tile_base = (int64_t)(c.tile_e - 1 - c.tile_b) * kTile;
    const int need = (int)(c.len - tile_base);                 // 1..kTile
    const int64_t nwords = (c.len + 31) >> 5;
    double a[kGroup], q[kGroup];
    unsigned cnan[kGroup], cinf[kGroup];
#pragma unroll
    for (int w = 0; w < kGroup; ++w) { a[w] = 0.0; q[w] = 0.0; cnan[w] = 0u; cinf[w] = 0u; }
    for (int e0 = 0; e0 < need; e0 += 128) {
        const int rem = need - e0 - 4 * lane;
        const int valid = rem >= 4 ? 4 : (rem > 0 ? rem : 0);
        const int64_t irel = tile_base + e0 + 4 * lane;
        uint32_t posR = 0u, negR = 0u;
        float acc[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
        for (int w = 0; w < kGroup; ++w) {
            if (w >= W) break;
            const float *row = p.g + (size_t)w * p.worker_stride + c.off + irel;
            float x[4] = {0.f, 0.f, 0.f, 0.f};
            if (valid == 4) {
                const float4 v = __ldcs(reinterpret_cast<const float4 *>(row));
                x[0] = v.x; x[1] = v.y; x[2] = v.z; x[3] = v.w;
            } else {
#pragma unroll
                for (int k = 0; k < 3; ++k)
                    if (k < valid) x[k] = __ldcs(row + k);
            }
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                const float v = x[k];
                if (c.isL || HEALTH) a[w] += (double)fabsf(v);
                if (HEALTH) {
                    if (v != v) ++cnan[w];
                    else if (fabsf(v) == INFINITY) ++cinf[w];
                    else q[w] += (double)v * (double)v;
                }
                if (c.isL) {
                    if (v > tau) posR |= (1u << k) << (4 * w);
                    if (ternary && v < ntau) negR |= (1u << k) << (4 * w);
                } else {
                    acc[k] = (w == 0) ? v : __fadd_rn(acc[k], v);
                }
            }
        }
        if (c.isL) {
            if (p.P) {
                const int64_t wi = (irel >> 5);                 // same word for the 8 lanes of an octet
                const bool stp = ((lane & 7) < W) && (wi < nwords) && (e0 + 32 * (lane >> 3) < need);
                const size_t o = (size_t)(lane & 7) * p.plane_stride + c.woff + wi;
                const uint32_t pw = nib_transpose8(posR, tctl);
                if (stp) p.P[o] = pw;
                if (ternary) {
                    const uint32_t nwd = nib_transpose8(negR, tctl);
                    if (stp) p.N[o] = nwd;
                }
            }
            const uint32_t d = ternary ? vote4<true>(posR, negR, W, p.margin) : vote4<false>(posR, negR, W, p.margin);
            if (valid > 0) p.dirs[(size_t)c.woff * 8 + (size_t)(irel >> 2)] = (uint8_t)d;
        } else {
            float *o = p.out + c.off + irel;
#pragma unroll
            for (int k = 0; k < 4; ++k)
                if (k < valid) o[k] = __fmul_rn(p.alpha, acc[k]);
        }
    }
#pragma unroll
    for (int w = 0; w < kGroup; ++w) {
        if (w >= W) break;
        const double da = warp_sum(a[w]);
        const size_t o = (size_t)w * T + c.t;
        if (HEALTH) {
            const double dq = warp_sum(q[w]);
            const unsigned n1 = warp_sum(cnan[w]), n2 = warp_sum(cinf[w]);
            if (lane == 0) {
                if (dq != 0.0) atomicAdd(p.sumsq + o, dq);
                if (n1) atomicAdd(p.nan_cnt + o, (unsigned long long)n1);
                if (n2) atomicAdd(p.inf_cnt + o, (unsigned long long)n2);
            }
        }
        if (lane == 0 && c.isL && da != 0.0) atomicAdd(p.abs_sum + o, da);
    }
}

extern __shared__ __align__(128) unsigned char smem_raw[];

// ---------------------------------------------------------------------------------------------
// the kernel
// ---------------------------------------------------------------------------------------------
template <bool HEALTH>
__global__ void __maxnreg__(96) fused_passA_kernel(const __grid_constant__ StreamParams p) {
    const PlanView pv = plan_view(p.plan, p.T);
    if (pv.hdr->magic != kPlanMagic || pv.hdr->status != NF_OK) return;
    constexpr int stages = kStages;
    const FusedSmem sm = carve(smem_raw, stages);
    const int n_tiles = pv.hdr->n_tiles;
    const int W = p.W;                          // 1..8: one worker group (launch_fused_passA)
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;

    if (tid == 0) {
        for (int s = 0; s < stages; ++s) { mbar_init(sm.full + s, 1); mbar_init(sm.empty + s, kCW); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    for (int i = tid; i < 256; i += kFThreads) { sm.nan[i] = 0u; sm.inf[i] = 0u; }
    for (int i = tid; i < kCW * 2 * W; i += kFThreads) sm.wacc[i] = 0.0;
    __syncthreads();

    // =========================================================================================
    // producer: one elected lane issues the bulk copies of every fast tile
    // =========================================================================================
    if (warp == kCW) {
        if (lane != 0) return;
        const uint64_t pol = policy_evict_first();
        int st = 0;
        uint32_t ph = 0;
        TensorCur c{};
        c.tile_e = 0;
        // full tiles of aligned tensors (the consumers walk exactly the same sequence)
        {
            for (int tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
                if (tile >= c.tile_e) tensor_lookup(p, pv, tile, c);
                if (!c.aligned || tile + 1 >= c.tile_e) continue;
                const float *src = p.g + c.off + (int64_t)(tile - c.tile_b) * kTile;
                mbar_wait(sm.empty + st, ph ^ 1u);
                mbar_expect_tx(sm.full + st, (uint32_t)(W * kTile * 4));
                float *dst = sm.ring + (size_t)st * kStageFloats;
                for (int w = 0; w < W; ++w)
                    bulk_g2s(dst + w * kTile, src + (size_t)w * p.worker_stride, (uint32_t)(kTile * 4), sm.full + st, pol);
                if (++st == stages) { st = 0; ph ^= 1u; }
            }
        }
        return;
    }
    // =========================================================================================
    // tail warp: last tile of every aligned tensor, tensors dealt round-robin over the CTAs
    // =========================================================================================
    if (warp == kCW + 1) {
        for (int t = blockIdx.x; t < p.T; t += gridDim.x) {
            TensorCur c;
            c.t = t;
            c.tile_b = __ldg(pv.tile_prefix + t);
            c.tile_e = __ldg(pv.tile_prefix + t + 1);
            if (c.tile_e == c.tile_b) continue;                  // empty tensor
            c.off = __ldg(p.off + t);
            c.len = __ldg(p.len + t);
            if (((c.off | p.worker_stride) & 3) != 0) continue;  // unaligned rows: LDG kernel
            c.isL = __ldg(p.route + t) == NF_ROUTE_L;
            c.woff = c.isL ? __ldg(p.woff + t) : 0;
            c.tau = (p.tau && c.isL) ? __ldg(p.tau + t) : 0.f;
            c.aligned = true;
            tail_tile_warp<HEALTH>(p, c, lane);
        }
        return;
    }

    // =========================================================================================
    // consumers
    // =========================================================================================
    const int ctid = tid;                       // 0..511
    const TCtl tctl = make_tctl(lane);
    const bool ternary = p.ternary != 0;
    const int tile_step = (int)gridDim.x;
    float af[8], qf[8];                         // FP32 partials of the current worker group
#pragma unroll
    for (int i = 0; i < 8; ++i) { af[i] = 0.f; qf[i] = 0.f; }
    int kcnt = 0, last_bulk = 0;
    int st = 0;
    uint32_t ph = 0;
    TensorCur c{};
    c.tile_e = 0;
    c.t = -1;
    bool touched = false;                       // this CTA accumulated something for tensor c.t
    bool fastT = false;                         // current tensor qualifies for the fast path
    uint32_t *pP = nullptr, *pN = nullptr;      // this thread's plane-word / direction / output slots
    uint8_t *pD = nullptr;                      //   of tile 0 of the current tensor
    float *pO = nullptr;

    auto flush_tensor = [&]() __attribute__((always_inline)) {
        if (kcnt > 0) { stat_flush<HEALTH>(p, sm, af, qf, c.off, c.len, c.tile_b, 0, W, kcnt, last_bulk, tile_step, ctid); kcnt = 0; }
        consumer_sync();
        for (int j = ctid; j < 2 * W; j += kCThreads) {
            double tot = 0.0;
#pragma unroll
            for (int k = 0; k < kCW; ++k) { tot += sm.wacc[(size_t)k * 2 * W + j]; sm.wacc[(size_t)k * 2 * W + j] = 0.0; }
            if (tot != 0.0) {
                const size_t o = (size_t)(j >> 1) * p.T + c.t;
                if ((j & 1) == 0) { if (c.isL) atomicAdd(p.abs_sum + o, tot); }
                else if (HEALTH) atomicAdd(p.sumsq + o, tot);
            }
        }
        if (HEALTH) {
            for (int w = ctid; w < W; w += kCThreads) {
                const unsigned cn_ = sm.nan[w], ci_ = sm.inf[w];
                const size_t o = (size_t)w * p.T + c.t;
                if (cn_) { atomicAdd(p.nan_cnt + o, (unsigned long long)cn_); sm.nan[w] = 0u; }
                if (ci_) { atomicAdd(p.inf_cnt + o, (unsigned long long)ci_); sm.inf[w] = 0u; }
            }
        }
        consumer_sync();
    };

    for (int tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
        if (tile >= c.tile_e) {
            if (touched) flush_tensor();
            tensor_lookup(p, pv, tile, c);
            touched = false;
            fastT = c.aligned;
            const size_t pl = (size_t)(lane & 7) * p.plane_stride + c.woff + warp * 4 + (lane >> 3);
            pP = (c.isL && p.P) ? p.P + pl : nullptr;
            pN = (c.isL && p.P && ternary) ? p.N + pl : nullptr;
            pD = c.isL ? p.dirs + (size_t)c.woff * 8 + ctid : nullptr;
            pO = p.out + c.off + 4 * ctid;
        }
        if (!fastT || tile + 1 >= c.tile_e) continue;                        // left to the LDG kernel
        {
            // ---- fast path: full tile, aligned rows, one worker group, data in the ring ----------
            const int rel = tile - c.tile_b;
            mbar_wait(sm.full + st, ph);
            const float *sb = sm.ring + (size_t)st * kStageFloats + 4 * ctid;
            uint64_t *const empty_bar = sm.empty + st;
            if (++st == stages) { st = 0; ph ^= 1u; }
            if (c.isL) {
                uint32_t posR = 0u, negR = 0u;
                const float tau = c.tau, ntau = -c.tau;
                if (ternary) {
                    if (W == kGroup) fast_signs<2, HEALTH, true>(sb, W, tau, ntau, af, qf, posR, negR);
                    else fast_signs<2, HEALTH, false>(sb, W, tau, ntau, af, qf, posR, negR);
                } else {
                    if (W == kGroup) fast_signs<1, HEALTH, true>(sb, W, tau, ntau, af, qf, posR, negR);
                    else fast_signs<1, HEALTH, false>(sb, W, tau, ntau, af, qf, posR, negR);
                }
                __syncwarp();
                if (lane == 0) mbar_arrive(empty_bar);
                if (pP) {
                    const bool stp = (lane & 7) < W;
                    const uint32_t pw = nib_transpose8(posR, tctl);
                    if (stp) pP[(size_t)rel * (kTile / 32)] = pw;
                    if (ternary) {
                        const uint32_t nwd = nib_transpose8(negR, tctl);
                        if (stp) pN[(size_t)rel * (kTile / 32)] = nwd;
                    }
                }
                const uint32_t d = ternary ? vote4<true>(posR, negR, W, p.margin) : vote4<false>(posR, negR, W, p.margin);
                pD[(size_t)rel * (kTile / 4)] = (uint8_t)d;
            } else {
                float4 r = (W == kGroup) ? fast_fp32<HEALTH, true>(sb, W, af, qf) : fast_fp32<HEALTH, false>(sb, W, af, qf);
                __syncwarp();
                if (lane == 0) mbar_arrive(empty_bar);
                r.x = __fmul_rn(p.alpha, r.x); r.y = __fmul_rn(p.alpha, r.y);
                r.z = __fmul_rn(p.alpha, r.z); r.w = __fmul_rn(p.alpha, r.w);
                __stcs(reinterpret_cast<float4 *>(pO + (size_t)rel * kTile), r);
            }
            touched = true;
            last_bulk = tile;
            if (++kcnt == kKTiles) { stat_flush<HEALTH>(p, sm, af, qf, c.off, c.len, c.tile_b, 0, W, kcnt, tile, tile_step, ctid); kcnt = 0; }
        }
    }
    if (touched) flush_tensor();

}

// ---------------------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------------------
template <bool HEALTH>
static cudaError_t launch_fused_t(const StreamParams &p, int64_t n, cudaStream_t s) {
    const size_t smem = fused_smem_bytes(kStages, kGroup);
    static bool configured = false;
    if (!configured) {
        cudaError_t e = cudaFuncSetAttribute(fused_passA_kernel<HEALTH>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        configured = true;
    }
    int64_t work = n / kTile > p.T ? n / kTile : p.T;        // full tiles (consumers) or tensors (tail warp)
    if (work <= 0) return cudaSuccess;
    int64_t grid = device_sm_count();                        // persistent: one CTA per SM
    if (grid > work) grid = work;
    fused_passA_kernel<HEALTH><<<(unsigned)grid, kFThreads, smem, s>>>(p);
    return cudaGetLastError();
}

// Full tiles of 16-byte-aligned tensors, W <= 8. The caller runs the LDG streaming kernel with
// skip_fast = 1 for the tensors whose rows are not 16-byte aligned.
cudaError_t launch_fused_passA(bool health, const StreamParams &p, int64_t n, cudaStream_t s) {
    if (p.W > kGroup) return cudaErrorInvalidValue;
    return health ? launch_fused_t<true>(p, n, s) : launch_fused_t<false>(p, n, s);
}

}  // namespace nf
