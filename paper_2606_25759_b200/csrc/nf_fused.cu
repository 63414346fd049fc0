// nf_fused.cu — the fused path of nf_aggregate_bucket after the route kernel: route-aware pack + sign
// count + majority vote + FP32-route sum + abs-sums + health statistics from ONE read of the W x n
// gradients (pass A) and the decode out = S_t * d (pass B), in one persistent kernel per bucket.
// PAPER §5.2, §3.3; SURVEY §8(a) a2/a3/a4a/a4b, §8(d) "fused floor".
//
// Blackwell design (HBM-bound streaming, no contraction -> no tensor cores), DESIGN.md §6:
//  * one persistent CTA per SM: 16 consumer warps, a producer warp, a housekeeping warp, 2 decode warps;
//  * the producer's elected lane takes tiles (2048 elements of one tensor) from a device-wide cursor and
//    streams them, 8 workers at a time (64 KB), from HBM into a 3-stage shared-memory ring with 1-D bulk
//    async copies (cp.async.bulk, the TMA engine) that complete on an mbarrier, with an L2 evict-first
//    policy (the gradients are read exactly once);
//  * consumer warps wait on the stage's "full" mbarrier, read one float4 per worker (conflict-free
//    LDS.128) and release the stage on its "empty" mbarrier;
//  * per thread: 4 consecutive elements of up to 8 workers -> one 4-bit nibble per worker in one
//    register per plane; counts are popcounts under a 0x11111111 mask; packed plane words come
//    from an 8x8 nibble transpose across 8 lanes;
//  * abs-sum / sum of squares: FP32 partials over kKTiles tiles (<= 16 elements, pairwise inside a
//    float4), FP32 warp reduce-scatter, FP64 per warp; a failed range check (NaN, Inf, FP32
//    over/underflow) sends the offending threads to an exact FP64 re-read of just those elements;
//  * ragged last tiles and tensors whose rows are not 16-byte aligned go through the same ring;
//  * each CTA publishes its finished tiles per tensor (release); decode warps, and the consumers once
//    the tiles are exhausted, acquire the per-tensor counter and expand the 2-bit directions.
#include <float.h>
#include <utility>
#include "nf_internal.cuh"

namespace nf {

constexpr int kCW = 16;                          // consumer warps
constexpr int kCThreads = kCW * 32;              // 512 threads x 4 elements = one tile
#ifndef NF_KDW
#define NF_KDW 2
#endif
#ifndef NF_KDU
#define NF_KDU 2
#endif
#ifndef NF_KKT
#define NF_KKT 4
#endif
#ifndef NF_KCHUNK
#define NF_KCHUNK 4                      // longest run of consecutive tiles one CTA takes at a time
#endif
constexpr int kDW = NF_KDW;                      // decode warps (pass B inside the kernel)
constexpr int kFThreads = kCThreads + 64 + kDW * 32;   // + producer warp + housekeeping warp + decode warps
constexpr int kDU = NF_KDU;                      // decode: units in flight per warp
constexpr int kPitch = kTile + 4;                // ring row: one tile of one worker + room for a misaligned head
constexpr int kStageFloats = kGroup * kPitch;    // 8 workers
constexpr int kStageBytes = kStageFloats * 4;    // 64 KB + 128 B
constexpr int kKTiles = NF_KKT;                  // tiles of FP32 partial accumulation (<= 4: exact_redo's list)
#ifndef NF_MRUN
#define NF_MRUN 4
#endif
constexpr int kMRun = NF_MRUN;                   // MULTI: tiles per group-major run (1 = tile-major order), <= kKTiles
static_assert(kMRun >= 1 && kMRun <= kKTiles && kMRun <= 4, "a run is flushed once: exact_redo lists <= 4 tiles");
constexpr int kMaxStages = 4;
constexpr int kStages = 3;                       // ring depth: 3 x 64 KB
static_assert(kTile == kCThreads * 4, "one float4 per consumer thread per worker and tile");

// named barriers 2 + b: hand-over of segment buffer b from the 16 consumer warps (arrive, never wait) to the reducer
// warp (sync: a hardware wait, no polling)
__device__ __forceinline__ void seg_bar_arrive(int b) { asm volatile("bar.arrive %0, %1;" ::"r"(2 + b), "n"(kCW * 32 + 32) : "memory"); }
__device__ __forceinline__ void seg_bar_sync(int b) { asm volatile("bar.sync %0, %1;" ::"r"(2 + b), "n"(kCW * 32 + 32) : "memory"); }
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
//   [0, 64)         mbarriers full[4], empty[4]
//   [64, 112)       per ring stage: tile index, run length (MULTI), end-of-segment flag
//   [128, 384)      scratch of the in-kernel routing scan
//   [416, 512)      segment buffers: mbarriers free[2]; [432, 448) aux words; the record handed over with each buffer [2][8]
//   [384, 416)      CTA-wide flags (init role, last arriver of a tensor, last CTA of the grid, decode chunk, pass A done)
//   [1024, 3072)    NaN / Inf tallies, 256 workers each
//   [3072, 4096)    per-worker scales s_w of the tensor being finalised, 256 floats
//   [4096, 8192)    decode table: byte of 4 (+,-) flag pairs -> float4 of directions in {-1, 0, +1}
//   [8192, 17408)   per-tensor metadata of the first kMetaCap tensors (tile prefix, off, len, woff, tau)
//   [17408, ...)    ring [stages][8][kPitch] floats
//   after the ring  per-warp FP64 totals {abs, sq} per worker of one record, [2][kCW][2*min(W, kRecW)] doubles: a
//                   segment is handed to the reducer warp in records of at most kRecW workers, double-buffered
// ---------------------------------------------------------------------------------------------
constexpr int kSmemMeta = 8192;
constexpr int kSmemHdr = kSmemMeta + 9216;       // 4*(cap+1) + 3*8*cap + 4*cap = 8196 bytes, padded
struct FusedSmem {
    float *ring;
    uint64_t *full, *empty;
    int *tile_of;                // [kMaxStages] tile held by a stage, -1 = no more tiles
    int *run_of;                 // [kMaxStages] MULTI: length R of the run of tiles the stage belongs to
    int *seg_of;                 // [kMaxStages] 1: the tile ends a segment (last tile of its scheduling unit or tensor)
    int *flag;                   // [8] CTA-wide flags
    int *aux;                    // [4] [0]: tiles of the previous bucket + 1 (0: not read yet)
    float *sw;                   // [256] per-worker scales of the tensor being finalised
    uint64_t *seg_free;          // [2] mbarriers: the reducer warp is through with a segment buffer
    int *seg_rec;                // [2][8] record handed over with a buffer: tensor (-1: no more), kind, route, tiles, ...
    unsigned int *nan, *inf;     // [256] each
    float4 *dtab;                // [256]
    int32_t *m_tile;             // [kMetaCap + 1] exclusive tile prefix
    int64_t *m_off, *m_len, *m_woff;   // [kMetaCap]; woff = -1 when the tensor is not low-bit routed
    float *m_tau;                // [kMetaCap]
    double *wacc;                // [2][kCW][2*min(W, kRecW)]
};
constexpr int kRecW = 32;                        // workers per record handed to the reducer warp
__host__ __device__ inline int fused_recw(int W) { return W < kRecW ? W : kRecW; }
__host__ __device__ inline size_t fused_smem_bytes(int stages, int W) {
    return (size_t)kSmemHdr + (size_t)stages * kStageBytes + sizeof(double) * kCW * 2 * (size_t)fused_recw(W) * 2;
}
__device__ __forceinline__ FusedSmem carve(unsigned char *base, int stages) {
    FusedSmem s;
    s.full = (uint64_t *)base;
    s.empty = s.full + kMaxStages;
    s.tile_of = (int *)(base + 64);
    s.run_of = (int *)(base + 80);
    s.seg_of = (int *)(base + 96);
    s.flag = (int *)(base + 384);
    s.aux = (int *)(base + 432);
    s.sw = (float *)(base + 3072);
    s.seg_free = (uint64_t *)(base + 416);
    s.seg_rec = (int *)(base + 448);
    s.nan = (unsigned int *)(base + 1024);
    s.inf = s.nan + 256;
    s.dtab = (float4 *)(base + 4096);
    s.m_off = (int64_t *)(base + kSmemMeta);
    s.m_len = s.m_off + kMetaCap;
    s.m_woff = s.m_len + kMetaCap;
    s.m_tau = (float *)(s.m_woff + kMetaCap);
    s.m_tile = (int32_t *)(s.m_tau + kMetaCap);
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
// Tensor of a tile. Buckets of up to kMetaCap tensors are served from the shared-memory copy the
// CTA made at start (a tensor change then costs a few LDS instead of a chain of L2 round trips).
__device__ __forceinline__ void tensor_lookup(const StreamParams &p, const PlanView &pv, const FusedSmem &sm, int tile,
                                              TensorCur &c) {
    if (p.T <= kMetaCap) {
        int lo = 0, hi = p.T;                    // invariant: m_tile[lo] <= tile < m_tile[hi]
        while (hi - lo > 1) {
            const int mid = (lo + hi) >> 1;
            if (sm.m_tile[mid] <= tile) lo = mid; else hi = mid;
        }
        c.t = lo;
        c.tile_b = sm.m_tile[lo];
        c.tile_e = sm.m_tile[lo + 1];
        c.off = sm.m_off[lo];
        c.len = sm.m_len[lo];
        const int64_t wo = sm.m_woff[lo];
        c.isL = wo >= 0;
        c.woff = c.isL ? wo : 0;
        c.tau = sm.m_tau[lo];
    } else {
        const int t = upper_tensor<int32_t>(pv.tile_prefix, p.T, tile);
        c.t = t;
        c.tile_b = __ldg(pv.tile_prefix + t);
        c.tile_e = __ldg(pv.tile_prefix + t + 1);
        c.off = __ldg(p.off + t);
        c.len = __ldg(p.len + t);
        c.isL = __ldg(p.route + t) == NF_ROUTE_L;
        c.woff = c.isL ? __ldg(p.woff + t) : 0;
        c.tau = (p.tau && c.isL) ? __ldg(p.tau + t) : 0.f;
    }
    c.aligned = (((c.off | p.worker_stride) & 3) == 0);
}
// Exact FP64 re-read of one thread's elements of worker `wg` over the last `cnt` (<= 4) tiles of the
// current tensor (`recent`, most recent first) (rare: NaN / Inf / FP32 range trouble in the FP32 partials). Returns
// {sum |x|, sum of x^2}, both over the FINITE x only; NaN / Inf are tallied in shared memory slot `slot` (the
// tensor's last arriver turns a non-zero tally into the IEEE result of the sum: NaN, else +Inf).
template <bool HEALTH>
__device__ __noinline__ double2 exact_redo(const float *__restrict__ g, int64_t worker_stride, int wg,
                                           int64_t off_t, int64_t len_t, int tile_b, int4 recent, int cnt, int ctid,
                                           unsigned int *s_nan, unsigned int *s_inf, int slot, bool aligned) {
    double da = 0.0, dq = 0.0;
    const float *row = g + (size_t)wg * worker_stride + off_t;
    // all loads first (independent, one round trip), then the arithmetic
    float x[4][4];
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        const int tl = j == 0 ? recent.x : (j == 1 ? recent.y : (j == 2 ? recent.z : recent.w));
        const int64_t base = (int64_t)(tl - tile_b) * kTile + 4 * ctid;
#pragma unroll
        for (int k = 0; k < 4; ++k) x[j][k] = 0.f;
        if (j < cnt) {
            if (aligned && base + 4 <= len_t) {
                const float4 v = __ldg(reinterpret_cast<const float4 *>(row + base));
                x[j][0] = v.x; x[j][1] = v.y; x[j][2] = v.z; x[j][3] = v.w;
            } else {
#pragma unroll
                for (int k = 0; k < 4; ++k)
                    if (base + k < len_t) x[j][k] = __ldg(row + base + k);
            }
        }
    }
    unsigned cn = 0u, ci = 0u;
#pragma unroll
    for (int j = 0; j < 4; ++j)
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            const float v = x[j][k];                         // padding zeros add nothing
            if (v != v) ++cn;
            else if (fabsf(v) == INFINITY) ++ci;
            else {
                da += (double)fabsf(v);
                if (HEALTH) dq += (double)v * (double)v;
            }
        }
    if (cn) atomicAdd(&s_nan[slot], cn);
    if (ci) atomicAdd(&s_inf[slot], ci);
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
// full tiles of a 16-byte-aligned tensor, one worker group of up to 8 workers, data in the ring
// ---------------------------------------------------------------------------------------------
// L tile: sign indicators of this thread's 4 elements of every worker (nibble w of posR / negR) and
// the FP32 abs / square partials. KIND 1 = G-Binary, 2 = G-Ternary.
template <int KIND, bool HEALTH, bool FULLW>
__device__ __forceinline__ void fast_signs(const float *sb, int nw, float tau, float ntau, float (&af)[8],
                                           float (&qf)[8], uint32_t &posR, uint32_t &negR) {
#pragma unroll
    for (int w = 0; w < kGroup; ++w) {
        if (!FULLW && w >= nw) break;
        const float4 v = *reinterpret_cast<const float4 *>(sb + w * kPitch);
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
__device__ __forceinline__ float4 fast_fp32(const float *sb, int nw, float (&af)[8], float (&qf)[8], float4 acc, bool first) {
#pragma unroll
    for (int w = 0; w < kGroup; ++w) {
        if (!FULLW && w >= nw) break;
        const float4 v = *reinterpret_cast<const float4 *>(sb + w * kPitch);
        if (HEALTH) {
            af[w] += (fabsf(v.x) + fabsf(v.y)) + (fabsf(v.z) + fabsf(v.w));
            qf[w] = fmaf(v.x, v.x, qf[w]); qf[w] = fmaf(v.y, v.y, qf[w]);
            qf[w] = fmaf(v.z, v.z, qf[w]); qf[w] = fmaf(v.w, v.w, qf[w]);
        }
        if (w == 0 && first) {
            acc = v;
        } else {
            acc.x = __fadd_rn(acc.x, v.x); acc.y = __fadd_rn(acc.y, v.y);
            acc.z = __fadd_rn(acc.z, v.z); acc.w = __fadd_rn(acc.w, v.w);
        }
    }
    return acc;
}
// Slow tiles, one instantiation with uniform branches on the tile kind:
//  * ragged last tile of an aligned tensor (need < kTile elements): the ring holds the whole float4s;
//    the one thread that owns the partial float4 reads its 1..3 elements from global memory;
//  * any tile of a tensor whose rows are NOT 16-byte aligned (unal): the producer copied every row
//    from the 16-byte boundary below it, so worker w's elements start m_w = (m0 + w*mstep) & 3
//    floats into its ring row and are read with scalar shared-memory loads.
// Threads past the end of the tensor see zeros.
template <bool HEALTH>
__device__ __forceinline__ void slow_tile(const float *sb, const float *grow, int64_t worker_stride, int nw, int valid,
                                          bool unal, int m0, int mstep,
                                            bool isL, bool ternary, float tau, float ntau, float (&af)[8],
                                            float (&qf)[8], uint32_t &posR, uint32_t &negR, float4 &acc, bool first) {
#pragma unroll
    for (int w = 0; w < kGroup; ++w) {
        if (w >= nw) break;
        float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
        if (unal) {
            const float *b = sb + w * kPitch + ((m0 + w * mstep) & 3);
            if (valid > 0) v.x = b[0];
            if (valid > 1) v.y = b[1];
            if (valid > 2) v.z = b[2];
            if (valid > 3) v.w = b[3];
        } else if (valid == 4) {
            v = *reinterpret_cast<const float4 *>(sb + w * kPitch);
        } else if (valid > 0) {
            const float *g = grow + (size_t)w * worker_stride;
            v.x = __ldg(g);
            if (valid > 1) v.y = __ldg(g + 1);
            if (valid > 2) v.z = __ldg(g + 2);
        }
        if (isL || HEALTH) {
            af[w] += (fabsf(v.x) + fabsf(v.y)) + (fabsf(v.z) + fabsf(v.w));
            if (HEALTH) {
                qf[w] = fmaf(v.x, v.x, qf[w]); qf[w] = fmaf(v.y, v.y, qf[w]);
                qf[w] = fmaf(v.z, v.z, qf[w]); qf[w] = fmaf(v.w, v.w, qf[w]);
            }
        }
        if (isL) {
            posR |= ((v.x > tau ? 1u : 0u) | (v.y > tau ? 2u : 0u) | (v.z > tau ? 4u : 0u) | (v.w > tau ? 8u : 0u)) << (4 * w);
            if (ternary)
                negR |= ((v.x < ntau ? 1u : 0u) | (v.y < ntau ? 2u : 0u) | (v.z < ntau ? 4u : 0u) | (v.w < ntau ? 8u : 0u)) << (4 * w);
        } else if (w == 0 && first) {
            acc = v;
        } else {
            acc.x = __fadd_rn(acc.x, v.x); acc.y = __fadd_rn(acc.y, v.y);
            acc.z = __fadd_rn(acc.z, v.z); acc.w = __fadd_rn(acc.w, v.w);
        }
    }
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

// FP32 partials of worker group [w0, w0+nw) over the last `cnt` bulk tiles (one segment) -> warp totals (FP32
// butterfly reduce-scatter) -> this warp's FP64 slots of the segment in shared memory (`wbuf`, stored, not
// added: a segment is reduced over the warps and leaves the CTA at once, see seg_reduce). Range check on the warp
// totals: |x| sums finite, squares neither over- nor underflowed; otherwise the warp re-reads
// exactly those elements in FP64 (and tallies NaN / Inf).
template <bool HEALTH>
__device__ __forceinline__ void stat_flush(const StreamParams &p, const FusedSmem &sm, double *wbuf, int tally0, float (&af)[8],
                                           float (&qf)[8], int64_t off_t, int64_t len_t, int tile_b, int w0, int nw,
                                           int cnt, int4 recent, int ctid, bool aligned) {
    // (wbuf, tally0: the record buffer and its NaN / Inf tallies, both indexed by worker - first worker of the record)
    const int lane = ctid & 31, warp = ctid >> 5, W = p.W, wr0 = w0 % kRecW;
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
    double *slot = wbuf + (size_t)warp * 2 * fused_recw(W) + (size_t)wr0 * 2;
    if (bad == 0u) {
        if ((lane & 1) == 0 && wl < nw) slot[wl * 2 + stat] = (double)r;
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
                    e = exact_redo<HEALTH>(p.g, p.worker_stride, w0 + w, off_t, len_t, tile_b, recent, cnt, ctid, sm.nan,
                                           sm.inf, tally0 + wr0 + w, aligned);
                const double ea = warp_sum(e.x), eq = warp_sum(e.y);
                if (lane == 0) { slot[w * 2] = ea; slot[w * 2 + 1] = eq; }
            } else if ((lane & 1) == 0 && wl == w) {
                slot[w * 2 + stat] = (double)r;
            }
        }
    }
#pragma unroll
    for (int i = 0; i < 8; ++i) { af[i] = 0.f; qf[i] = 0.f; }
    __syncwarp();
}

// debug aid (nf_debug_trace): globaltimer stamps per CTA: 5 kernel entry, 6 after griddepcontrol.wait, 7 after the
// grid barrier of the in-kernel routing, 0 consumers start, 1 tiles exhausted, 2 last flush, 3 consumers' decode
// done, 4 decode warp done
__device__ __forceinline__ void trace_stamp(const StreamParams &p, int slot) {
    if (p.trace) {
        unsigned long long t;
        asm volatile("mov.u64 %0, %globaltimer;" : "=l"(t));
        p.trace[(size_t)blockIdx.x * 16 + slot] = t;
    }
}

// A bounded wait ran out (a lost CTA, a corrupted plan): report NF_ERR_CUDA through summary[NF_SUM_STATUS] and the
// plan instead of hanging or trapping, and drop the clean token so that the next call re-initialises the plan.
__device__ __noinline__ void report_timeout(const StreamParams &p) {
    PlanHeader *hdr = (PlanHeader *)p.plan;
    hdr->status = NF_ERR_CUDA;
    hdr->sched = 0ull;
    if (p.summary) p.summary[NF_SUM_STATUS] = NF_ERR_CUDA;
    __threadfence();
}

__device__ __forceinline__ unsigned long long ld_acquire_u64(const unsigned long long *p) {
    unsigned long long v;
    asm volatile("ld.acquire.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_release_u64(unsigned long long *p, unsigned long long v) {
    asm volatile("st.release.gpu.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}

// ---------------------------------------------------------------------------------------------
// pass B inside the kernel: out[off_t+i] = S_t * d for the low-bit tiles, as soon as tensor t is complete and
// finalised (plan.fin[t] != 0: every CTA's tiles of t are published and the tensor's last arriver has rounded
// the totals and computed S_t). A unit is half a tile (1024 elements), handed out in tile order by a
// device-wide cursor, so the wait is always on the earliest unfinished tensor. The dedicated decode warps
// overlap their stores with the consumers' reads of later tensors; the consumers join when their own tiles are
// done. Every store instruction writes 512 contiguous bytes.
// ---------------------------------------------------------------------------------------------
struct DecodeCur {
    int t_cur, tile_b, tile_e;
    int64_t off_t, len_t, woff_t;
    bool dec;
    float S_t;
};
// Units a decode warp hands on to the next kernel of the step when its CTA leaves (`stop`): every decode warp of the
// grid owns kHandOn entries of the plan's orph[] (unit + 1, 0 = empty; entries of CTA c, decode warp d at
// (c * kDW + d) * kHandOn), written with plain stores and read, then cleared, by the same warp of the next kernel:
// no atomics, no round trip before the CTA can go.
constexpr int kHandOn = 4;                       // <= 2 spans of kDU units in hand (the current one, the prefetched one)
struct HandOn {
    const volatile int *stop;                    // shared memory: this CTA takes no more units (NULL: never)
    int32_t *slots;                              // this warp's entries (NULL: hand nothing on, wait instead)
    int n;                                       // entries used so far
};
// where the units of a bucket come from: this kernel's own bucket (metadata in shared memory when T <= kMetaCap)
// or the previous bucket of the step (everything from global memory)
struct DecodeSrc {
    int T, n_tiles;
    bool smem_meta;
    const int32_t *tile_prefix;
    const int64_t *off, *len, *woff;
    const uint8_t *route;
    const unsigned long long *fin;
    const uint8_t *dirs;
    float *out;
    PlanHeader *hdr;
    int32_t *orph;
};
// A span = kDU consecutive units, by one warp, in two phases so that a warp can have the loads of its next span in
// flight while it stores the current one: decode_load (tensor lookup, wait for the tensor's scale, direction words)
// and decode_store (expand and write).
struct DecodeSpan {
    uint32_t dv[kDU][2];
    int64_t obase[kDU], rem[kDU];
    float S[kDU];
};
// `ho` (or NULL): once its stop flag is set (this CTA leaves the rest of the bucket's pass B to the next kernel of the
// step), units in hand that have not been started are not decoded any more, let alone waited for (the CTA would hold
// its SM for nothing until a tensor's last arriver, somewhere else, is through): they are handed on.
__device__ __forceinline__ void decode_load(const StreamParams &p, const DecodeSrc &src, const FusedSmem &sm, DecodeCur &dc,
                                            int u0, int u_lim, int lane, DecodeSpan &sp, HandOn *ho = nullptr) {
#pragma unroll
    for (int k = 0; k < kDU; ++k) {
        const int u = u0 + k;
        sp.rem[k] = 0; sp.obase[k] = 0; sp.S[k] = 0.f; sp.dv[k][0] = 0u; sp.dv[k][1] = 0u;
        if (u >= u_lim) continue;
        if (ho && ho->slots && ho->n < kHandOn && *ho->stop) {
            if (lane == 0) ho->slots[ho->n] = u + 1;
            ++ho->n;
            continue;
        }
        const int tile = u >> 1;
        if (tile >= dc.tile_e || tile < dc.tile_b) {             // (handed-on units do not come in tile order)
            if (src.smem_meta) {
                int lo = 0, hi = src.T;                  // invariant: m_tile[lo] <= tile < m_tile[hi]
                while (hi - lo > 1) {
                    const int mid = (lo + hi) >> 1;
                    if (sm.m_tile[mid] <= tile) lo = mid; else hi = mid;
                }
                dc.t_cur = lo; dc.tile_b = sm.m_tile[lo]; dc.tile_e = sm.m_tile[lo + 1];
                dc.off_t = sm.m_off[lo]; dc.len_t = sm.m_len[lo];
                dc.woff_t = sm.m_woff[lo];
                dc.dec = dc.woff_t >= 0;
            } else {
                const int t = upper_tensor<int32_t>(src.tile_prefix, src.T, tile);
                dc.t_cur = t; dc.tile_b = __ldg(src.tile_prefix + t); dc.tile_e = __ldg(src.tile_prefix + t + 1);
                dc.off_t = __ldg(src.off + t); dc.len_t = __ldg(src.len + t);
                dc.dec = __ldcg(src.route + t) == NF_ROUTE_L;
                dc.woff_t = dc.dec ? __ldcg(src.woff + t) : 0;
            }
            if (dc.dec) {
                // wait for the tensor's last arriver (it runs in a resident CTA, and so does every CTA that still
                // holds tiles of the tensor: nobody waits for a CTA that has not started)
                const unsigned long long *fp = src.fin + dc.t_cur;
                unsigned long long seen;
                bool handed = false;
                for (unsigned spins = 0;; ++spins) {
                    seen = ld_acquire_u64(fp);
                    if (seen) break;
                    if (ho && ho->slots && ho->n < kHandOn && *ho->stop) { handed = true; break; }
                    __nanosleep(100);
                    if (spins > (1u << 25)) { report_timeout(p); dc.dec = false; break; }   // > 4 s: give up loudly
                }
                if (handed) {
                    if (lane == 0) ho->slots[ho->n] = u + 1;
                    ++ho->n;
                    dc.tile_e = 0;                           // (nothing is known of this tensor: look again next time)
                    dc.tile_b = 0;
                    continue;
                }
                dc.S_t = __uint_as_float((uint32_t)seen);
            }
        }
        if (!dc.dec) continue;
        const int64_t wbase = (int64_t)(tile - dc.tile_b) * kTile + (u & 1) * 1024;     // tensor-relative
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            const int64_t i = wbase + h * 512 + lane * 16;
            if (i < dc.len_t)
                sp.dv[k][h] = __ldcg(reinterpret_cast<const uint32_t *>(src.dirs + (size_t)dc.woff_t * 8 + (size_t)(i >> 2)));
        }
        sp.obase[k] = dc.off_t + wbase;
        sp.rem[k] = dc.len_t - wbase;
        sp.S[k] = dc.S_t;
    }
}
__device__ __forceinline__ void decode_store(const DecodeSrc &src, const FusedSmem &sm, int lane, const DecodeSpan &sp) {
    const float4 *dtab = sm.dtab;
#pragma unroll
    for (int k = 0; k < kDU; ++k) {
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            const int64_t rh = sp.rem[k] - h * 512;
            if (rh <= 0) continue;                       // warp-uniform
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                // store j covers elements j*128 + lane*4 .. +3: direction byte (j*32 + lane)
                const uint32_t w32 = __shfl_sync(0xffffffffu, sp.dv[k][h], j * 8 + (lane >> 2));
                const uint32_t d = (w32 >> (8 * (lane & 3))) & 0xffu;
                const int64_t e0 = j * 128 + lane * 4;
                const int64_t r = rh - e0;
                if (r <= 0) continue;
                float4 v = dtab[d];
                v.x = __fmul_rn(sp.S[k], v.x); v.y = __fmul_rn(sp.S[k], v.y);
                v.z = __fmul_rn(sp.S[k], v.z); v.w = __fmul_rn(sp.S[k], v.w);
                float *o = src.out + sp.obase[k] + h * 512 + e0;
                if (r >= 4 && (sp.obase[k] & 3) == 0) {
                    __stcs(reinterpret_cast<float4 *>(o), v);
                } else {
                    o[0] = v.x;
                    if (r > 1) o[1] = v.y;
                    if (r > 2) o[2] = v.z;
                    if (r > 3) o[3] = v.w;
                }
            }
        }
    }
}
__device__ __forceinline__ void decode_span(const StreamParams &p, const DecodeSrc &src, const FusedSmem &sm, DecodeCur &dc,
                                            int u0, int u_lim, int lane) {
    DecodeSpan sp;
    decode_load(p, src, sm, dc, u0, u_lim, lane, sp);
    decode_store(src, sm, lane, sp);
}
// A dedicated decode warp: one span (kDU units) per trip to the bucket's cursor, the next trip issued before the span
// is processed (its round trip hides behind the span's loads and stores). More in flight per warp (2 or 4 spans per
// trip, or the next span's loads ahead of the current span's stores) made every config slower: the decode warps then
// take issue slots and L2 bandwidth the consumers need. `stop` (shared memory, or NULL): once it is set the warp
// takes no further units (what it holds it finishes): the rest is left to the next kernel of the step.
#ifndef NF_DSPANS
#define NF_DSPANS 1
#endif
// Returns whether the warp saw the cursor exhausted (false: it left because of `stop`).
__device__ __forceinline__ bool decode_warp_loop(const StreamParams &p, const DecodeSrc &src, const FusedSmem &sm,
                                                 const volatile int *stop, bool hand_on, volatile int *hint, int lane, int dwarp) {
    constexpr int kGU = NF_DSPANS * kDU;                    // units per trip
    const int total_units = src.n_tiles * 2;
    DecodeCur dc{-1, 0, 0, 0, 0, 0, false, 0.f};
    // (a grid beyond the list's capacity: the warps of the CTAs past it wait for their tensors instead)
    const int my_slot = ((int)blockIdx.x * kDW + dwarp) * kHandOn;
    HandOn ho{stop, (stop && hand_on && my_slot + kHandOn <= kMaxOrphans) ? src.orph + my_slot : nullptr, 0};
    constexpr int kStopped = 0x7fffffff;
    auto grab = [&]() -> int {
        int ub = kStopped;
        if (!(stop && *stop) && lane == 0) ub = atomicAdd(&src.hdr->unit_cursor, kGU);
        return ub;                                          // (lane 0's value is the one that counts)
    };
    int ub = __shfl_sync(0xffffffffu, grab(), 0);
    while (ub < total_units) {
        const int ub_next = grab();                         // in flight while this trip's spans are processed
        DecodeSpan sp[NF_DSPANS];
#pragma unroll
        for (int k = 0; k < NF_DSPANS; ++k) decode_load(p, src, sm, dc, ub + k * kDU, total_units, lane, sp[k], &ho);
#pragma unroll
        for (int k = 0; k < NF_DSPANS; ++k) decode_store(src, sm, lane, sp[k]);
        ub = __shfl_sync(0xffffffffu, ub_next, 0);
        if (lane == 0 && hint && ub != kStopped) *hint = ub;      // (where the cursor stands: the consumers size their first chunk by it)
    }
    return ub != kStopped;
}
// The consumers once their tiles are exhausted: ONE trip to the cursor per CTA and chunk (a few thousand warps
// arriving together on one address serialise: 15 us for the last warp served), chunk sizes guided by what is
// left (4 spans .. 16 spans per warp), spans dealt to the 16 warps round-robin.
__device__ __forceinline__ void decode_cta_loop(const StreamParams &p, const DecodeSrc &src, const FusedSmem &sm, int ctid,
                                                int cursor_hint) {
    const int total_units = src.n_tiles * 2, lane = ctid & 31, warp = ctid >> 5;
    DecodeCur dc{-1, 0, 0, 0, 0, 0, false, 0.f};
    // first chunk: an even share of what was left when this CTA's decode warps last looked (a backlog of many units is
    // then taken in one trip per CTA), at least 8 spans
    int chunk = kDU * min(max((total_units - cursor_hint) / ((int)gridDim.x * kDU), 8), 16 * kCW);
    for (;;) {
        if (ctid == 0) { sm.flag[3] = atomicAdd(&src.hdr->unit_cursor, chunk); sm.flag[6] = chunk; }
        consumer_sync();
        const int base = sm.flag[3];
        chunk = sm.flag[6];                                  // (ctid 0's: the hint the first chunk is sized by is racy)
        if (base >= total_units) break;
        const int lim = min(base + chunk, total_units);
        for (int u0 = base + kDU * warp; u0 < lim; u0 += kDU * kCW) decode_span(p, src, sm, dc, u0, lim, lane);
        if (lim >= total_units) break;                      // this chunk reached the end: no trip to find that out
        const int spans = (total_units - lim) / (2 * (int)gridDim.x * kDU);     // guided: half of an even share
        chunk = kDU * min(max(spans, 4), 16 * kCW);
        consumer_sync();                                    // everybody has read flag[3]
    }
}
// the same vote from byte-packed running counts (W > 8: several worker groups per tile)
__device__ __forceinline__ uint32_t vote4_packed(uint32_t cp, uint32_t cn, bool ternary, int W, int margin) {
    uint32_t d = 0u;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        const int c_p = (cp >> (8 * j)) & 0xff;
        const int c_n = ternary ? (int)((cn >> (8 * j)) & 0xff) : W - c_p;
        const int D = c_p - c_n;
        if (D > margin) d |= 1u << j;
        if (D < -margin) d |= 16u << j;
    }
    return d;
}

extern __shared__ __align__(128) unsigned char smem_raw[];

// The self-cleaning state of a bucket whose decode tail was drained by a later kernel, back to "clean" (by one warp,
// once nothing uses the state any more). The hand-on entries were cleared by whoever took them.
__device__ __forceinline__ void reset_bucket_state(void *plan, int T, int W, int lane) {
    const PlanView v = plan_view(plan, T);
    PlanHeader *h = (PlanHeader *)plan;
    for (int t = lane; t < T; t += 32) { v.done[t] = 0; v.fin[t] = 0ull; }
    if (lane == 0) {
        h->unit_cursor = 0;
        h->finish_count = 0;
        h->sched = (unsigned long long)clean_token(T, W) << 32;
    }
}

// A chained kernel's accounting for the PREVIOUS bucket of the step, whose decode tail it drains. Only the LAST kernel of
// a chain needs it: in the middle of a chain the state of bucket k-1 is reset by kernel k+1 (whose dependency wait on
// kernel k, which waited on kernel k-1, proves that nothing uses it any more), without any counting. Called by a whole
// warp that is through with that bucket: its cursor is exhausted (every unit has a taker) and what the warp took it has
// written. The parties of a CTA are its decode warps and, only if they registered as helpers before any decode warp
// was through (sm.flag[5] = helpers << 8 | parties through), its consumers. The CTA's last party counts the CTA in the
// previous bucket's plan, and the grid's last CTA resets that bucket's self-cleaning state. For the decode warps this
// happens early in the kernel, on nobody's critical path: a chained kernel ends without a device-wide round trip.
__device__ __forceinline__ void through_with_prev(const StreamParams &p, PlanHeader *prev_hdr, const PlanView &ppv,
                                                  const FusedSmem &sm, int lane) {
    __syncwarp();
    int last_party = 0;
    if (lane == 0) {
        const int old = atomicAdd(sm.flag + 5, 1);
        last_party = ((old & 0xff) + 1 == kDW + (old >> 8)) ? 1 : 0;
    }
    if (!__shfl_sync(0xffffffffu, last_party, 0)) return;
    int last = 0;
    if (lane == 0) last = atomicAdd(&prev_hdr->finish_count, 1) == (int)gridDim.x - 1;
    if (!__shfl_sync(0xffffffffu, last, 0)) return;
    reset_bucket_state(p.prev_plan, p.prev_T, p.prev_W, lane);
}


// ---------------------------------------------------------------------------------------------
// The tensor's last arriver (the CTA whose publication completed done[t]) rounds the exact totals of tensor t
// to FP64 once, writes abs_sum / sumsq / nan_cnt / inf_cnt, clears the accumulator slots for the next call,
// computes S_t = (float)(sum_w (double)(float)(A_w / len_t) / W) in worker order ("mean-absolute
// scale"; readings #7, #8) and publishes it: fin[t] = {1, S_t} releases the decode warps of every CTA.
// Done by ONE warp (the CTA's reducer warp), so that the consumers never stop for it.
//  * W <= 32: lane k holds word k of a worker's slot (one coalesced 256-byte load per worker, the loads of up to 8
//    workers in flight together), carries and rounding by shuffles;
//  * wider fan-in: lane = worker, 32 workers per pass, each lane walking its own slot (acc_round).
// ---------------------------------------------------------------------------------------------
// Eight workers' accumulators of tensor t, [w0, w0 + 8), rounded and written by ONE warp: lane k holds word k of each
// worker's slot (eight coalesced 256-byte loads in flight together), carries by shuffles, the 16 roundings by 16 lanes
// at once. Leaves sm.sw[w] = (float)(A_w / len_t) for the scale.
template <bool HEALTH>
__device__ __forceinline__ void finalize8(const StreamParams &p, const PlanView &pv, const FusedSmem &sm, int t, int64_t len_t,
                                          bool isL, bool read, int w0, int lane) {
    const int W = p.W, T = p.T;
    unsigned long long v[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        v[i] = 0ull;
        if (read && w0 + i < W) v[i] = __ldcg(pv.acc + ((size_t)(w0 + i) * T + t) * kAccWords + lane);
    }
    // (the clearing stores come after ALL the loads have been issued: a store behind a load of the same word
    // would serialise the eight round trips)
#pragma unroll
    for (int i = 0; i < 8; ++i)
        if (read && w0 + i < W) __stcg(pv.acc + ((size_t)(w0 + i) * T + t) * kAccWords + lane, 0ull);
    // the eight workers' carry chains and roundings are walked together (independent shuffle chains overlap)
    unsigned long long cn[8], ci[8], lo[8], hi[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        cn[i] = __shfl_sync(0xffffffffu, v[i], kAccNan);
        ci[i] = __shfl_sync(0xffffffffu, v[i], kAccInf);
        lo[i] = lane >= kAccNan ? 0ull : (v[i] & 0xffffffffull);
        hi[i] = lane >= kAccNan ? 0ull : (v[i] >> 32);
    }
    for (;;) {                                   // deferred carries ripple up (no carry into lanes 0 / kAccSq)
        bool more = false;
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            unsigned long long c = __shfl_up_sync(0xffffffffu, hi[i], 1);
            if (lane == kAccAbs || lane == kAccSq) c = 0ull;
            const unsigned long long x = lo[i] + c;
            lo[i] = x & 0xffffffffull;
            hi[i] = x >> 32;
            more |= hi[i] != 0ull;
        }
        if (!__any_sync(0xffffffffu, more)) break;
    }
    // The 16 roundings (8 workers x {sum |x|, sum x^2}) are done by 16 lanes AT ONCE, lane q = (worker q >> 1,
    // statistic q & 1): each lane fetches the three leading digits of its own accumulator from the lanes that
    // hold them and rounds once. (One after the other, by the whole warp, they were a chain of a few thousand
    // dependent instructions: 25 - 30 us for a warp that competes with 16 busy consumer warps, during which the
    // tensor's decode could not start.)
    uint32_t dg[8];
    unsigned nzb[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        dg[i] = (uint32_t)lo[i];
        nzb[i] = __ballot_sync(0xffffffffu, dg[i] != 0u);
    }
    const int wi = (lane & 15) >> 1, stat = lane & 1;
    const int l0 = stat ? kAccSq : kAccAbs, nwords = stat ? kAccSqWords : kAccAbsWords;
    unsigned my_nz = 0u;
    unsigned long long my_cn = 0ull, my_ci = 0ull;
#pragma unroll
    for (int i = 0; i < 8; ++i)
        if (wi == i) { my_nz = nzb[i]; my_cn = cn[i]; my_ci = ci[i]; }
    const unsigned m = (my_nz >> l0) & ((1u << nwords) - 1u);
    const int top = m ? 31 - __clz(m) : 0;
    const int s0 = l0 + top, s1 = l0 + max(top - 1, 0), s2 = l0 + max(top - 2, 0);
    unsigned long long d0 = 0ull, d1 = 0ull, d2 = 0ull;
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        const uint32_t a = __shfl_sync(0xffffffffu, dg[i], s0), b = __shfl_sync(0xffffffffu, dg[i], s1),
                       c = __shfl_sync(0xffffffffu, dg[i], s2);
        if (wi == i) { d0 = a; d1 = b; d2 = c; }
    }
    double val = 0.0;                            // the same arithmetic as warp_acc_round()
    if (m != 0u) {
        const unsigned long long hi64 = (d0 << 32) | (top >= 1 ? d1 : 0ull);
        const unsigned long long lo32 = top >= 2 ? d2 : 0ull;
        const bool sticky = top >= 3 && (m & ((1u << (top - 2)) - 1u)) != 0u;
        const int lz = __clzll((long long)hi64);
        unsigned long long mant = lz ? ((hi64 << lz) | (lo32 >> (32 - lz))) : hi64;
        if (sticky || ((lo32 << lz) & 0xffffffffull)) mant |= 1ull;
        val = scalbn(__ull2double_rn(mant), (stat ? kAccSqBase : kAccAbsBase) + 32 * top + 31 - lz - 63);
    }
    if (lane < 16 && w0 + wi < W) {
        const size_t o = (size_t)(w0 + wi) * T + t;
        if (stat == 0) {
            double a = 0.0;                                // 0 for tensors that are not low-bit routed
            if (read && isL) {
                a = val;
                if (my_cn) a = __longlong_as_double(0x7ff8000000000000ll);      // IEEE: a NaN term makes the sum NaN,
                else if (my_ci) a = __longlong_as_double(0x7ff0000000000000ll); // an Inf term (no NaN) makes it +Inf
            }
            p.abs_sum[o] = a;
            sm.sw[w0 + wi] = (float)(a / (double)len_t);
        } else if (HEALTH) {
            p.sumsq[o] = read ? val : 0.0;
            p.nan_cnt[o] = my_cn;
            p.inf_cnt[o] = my_ci;
        }
    }
}

template <bool HEALTH>
__device__ __noinline__ void finalize_tensor_warp(const StreamParams &p, const PlanView &pv, const FusedSmem &sm, int t,
                                                  int64_t len_t, bool isL, int lane) {
    const int W = p.W, T = p.T;
    const bool read = isL || HEALTH;
    if (W <= 32) {
        for (int w0 = 0; w0 < W; w0 += 8) finalize8<HEALTH>(p, pv, sm, t, len_t, isL, read, w0, lane);
    } else {
        for (int w = lane; w < W; w += 32) {
            const size_t o = (size_t)w * T + t;
            double A = 0.0;
            if (read) {
                unsigned long long wd[kAccWords];
                ulonglong2 *slot = reinterpret_cast<ulonglong2 *>(pv.acc + o * kAccWords);
#pragma unroll
                for (int i = 0; i < kAccWords / 2; ++i) {
                    const ulonglong2 x = __ldcg(slot + i);
                    wd[2 * i] = x.x;
                    wd[2 * i + 1] = x.y;
                }
#pragma unroll
                for (int i = 0; i < kAccWords / 2; ++i) __stcg(slot + i, make_ulonglong2(0ull, 0ull));
                const unsigned long long cn = wd[kAccNan], ci = wd[kAccInf];
                if (isL) {
                    A = acc_round(wd + kAccAbs, kAccAbsWords, kAccAbsBase);
                    if (cn) A = __longlong_as_double(0x7ff8000000000000ll);
                    else if (ci) A = __longlong_as_double(0x7ff0000000000000ll);
                }
                if (HEALTH) {
                    p.sumsq[o] = acc_round(wd + kAccSq, kAccSqWords, kAccSqBase);
                    p.nan_cnt[o] = cn;
                    p.inf_cnt[o] = ci;
                }
            }
            p.abs_sum[o] = A;
            sm.sw[w] = (float)(A / (double)len_t);
        }
    }
    if (!isL) return;
    __syncwarp();
    if (lane == 0) {
        double s = 0.0;
        for (int w = 0; w < W; ++w) s += (double)sm.sw[w];
        const float S = (float)(s / (double)W);
        pv.scale[t] = S;
        if (p.scale_out) p.scale_out[t] = S;
        st_release_u64(pv.fin + t, (1ull << 32) | (unsigned long long)__float_as_uint(S));    // (release: a fence of its own)
    }
    __syncwarp();
}

// The same by the CTA's 16 consumer warps, a warp per worker (used at the end of the kernel, when the consumers have
// nothing else to do and the tensor's decode is the critical path). Called by all consumer threads.
template <bool HEALTH>
__device__ __noinline__ void finalize_tensor(const StreamParams &p, const PlanView &pv, const FusedSmem &sm, int t,
                                             int64_t len_t, bool isL, int ctid) {
    const int W = p.W, T = p.T, warp = ctid >> 5, lane = ctid & 31;
    // wide fan-in: a warp per 8 workers, their loads in flight together (a warp per worker walks W / 16 slots one after
    // the other: 16 us at W = 64 between the last tile and the tensor's decode)
    if (W > kCW)
        for (int w0 = warp * 8; w0 < W; w0 += kCW * 8) finalize8<HEALTH>(p, pv, sm, t, len_t, isL, isL || HEALTH, w0, lane);
    for (int w = warp; w < W && W <= kCW; w += kCW) {          // a warp per worker: lane k holds word k of the slot
        const size_t o = (size_t)w * T + t;
        double A = 0.0;
        if (isL || HEALTH) {
            unsigned long long *slot = pv.acc + o * kAccWords;
            const unsigned long long v = __ldcg(slot + lane);
            __stcg(slot + lane, 0ull);
            const unsigned long long cn = __shfl_sync(0xffffffffu, v, kAccNan), ci = __shfl_sync(0xffffffffu, v, kAccInf);
            uint32_t digit;
            warp_acc_digits(v, lane, digit);
            const unsigned nz = __ballot_sync(0xffffffffu, digit != 0u);
            if (isL) {
                A = warp_acc_round(digit, nz, kAccAbs, kAccAbsWords, kAccAbsBase);
                if (cn) A = __longlong_as_double(0x7ff8000000000000ll);          // IEEE: a NaN term makes the sum NaN,
                else if (ci) A = __longlong_as_double(0x7ff0000000000000ll);     // an Inf term (no NaN) makes it +Inf
            }
            if (HEALTH) {
                const double Q = warp_acc_round(digit, nz, kAccSq, kAccSqWords, kAccSqBase);
                if (lane == 0) { p.sumsq[o] = Q; p.nan_cnt[o] = cn; p.inf_cnt[o] = ci; }
            }
        }
        if (lane == 0) {
            p.abs_sum[o] = A;                                  // 0 for tensors that are not low-bit routed
            sm.sw[w] = (float)(A / (double)len_t);
        }
    }
    if (!isL) return;                                      // CTA-uniform
    consumer_sync();
    if (ctid == 0) {
        double s = 0.0;
        for (int w = 0; w < W; ++w) s += (double)sm.sw[w];
        const float S = (float)(s / (double)W);
        pv.scale[t] = S;
        if (p.scale_out) p.scale_out[t] = S;
        st_release_u64(pv.fin + t, (1ull << 32) | (unsigned long long)__float_as_uint(S));    // (release: a fence of its own)
    }
}

// ---------------------------------------------------------------------------------------------
// the kernel
// ---------------------------------------------------------------------------------------------
#ifndef NF_TAIL4
#define NF_TAIL4 2                        // the last NF_TAIL4 x grid tiles are not handed out 4 at a time
#endif
#ifndef NF_TAIL4_M
#define NF_TAIL4_M 6                      // the same for W > 8, where a tile is W / 8 ring stages: no single-tile units
#endif
#ifndef NF_TAIL2_M
#define NF_TAIL2_M 0
#endif
#ifndef NF_GRAB
#define NF_GRAB 1                         // most scheduling units a producer takes per trip to the cursor
#endif
#ifndef NF_TAIL2
#define NF_TAIL2 1                        // the last NF_TAIL2 x grid tiles are handed out one at a time
#endif

template <bool HEALTH, bool MULTI>
__global__ void __maxnreg__(96) fused_passA_kernel(const __grid_constant__ StreamParams p, const int stages_arg) {
    const int stages = MULTI ? stages_arg : kStages;     // W <= 8: compile-time ring depth
    const FusedSmem sm = carve(smem_raw, stages);
    const int W = p.W;                          // MULTI: W > 8, several worker groups of 8 per tile
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    // Chaining (nf_aggregate_step), see the comment at the decode warps below. A chained kernel needs nothing of the
    // previous grid for its pass A and lets its own successor go at once; a kernel whose successor is chained lets
    // it go only after its own dependency wait, so that "everything before the step" is complete for the whole chain.
    if (!p.next_chained) pdl_launch_dependents();
    if (tid == 0) trace_stamp(p, 5);
    // A chained kernel reads its bucket's layout at once: like the gradients, it was complete before the step was
    // enqueued (nf.h), and the step's first kernel has waited for that. The round trip overlaps the set-up below.
    const bool early_meta = p.chained && p.inkernel_route;
    long long m_o = 0, m_l = 0, m_pe = 0;
    int m_el = 0;
    float m_tau = 0.f;
    if (early_meta && tid < p.T) {
        m_o = __ldg(p.off + tid);
        m_l = __ldg(p.len + tid);
        m_pe = tid == 0 ? 0 : __ldg(p.off + tid - 1) + __ldg(p.len + tid - 1);
        m_el = __ldg(p.elig + tid);
        if (p.tau) m_tau = __ldg(p.tau + tid);
    }

    if (tid == 0) {
        for (int s = 0; s < stages; ++s) { mbar_init(sm.full + s, 1); mbar_init(sm.empty + s, kCW); }
        for (int b = 0; b < 2; ++b) mbar_init(sm.seg_free + b, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    for (int i = tid; i < 256; i += kFThreads) { sm.nan[i] = 0u; sm.inf[i] = 0u; }
    if (tid < 8) sm.flag[tid] = 0;
    if (tid < 4) sm.aux[tid] = 0;
    for (int i = tid; i < 256; i += kFThreads)
        sm.dtab[i] = make_float4((float)((i & 1) - ((i >> 4) & 1)), (float)(((i >> 1) & 1) - ((i >> 5) & 1)),
                                 (float)(((i >> 2) & 1) - ((i >> 6) & 1)), (float)(((i >> 3) & 1) - ((i >> 7) & 1)));
    // warm the L2 with the small arrays the start-up chain reads (prefetches only: nothing the previous kernel on
    // the stream may still be writing is READ before the dependency wait). Every bucket has its own plan and
    // metadata, touched once per step: without this each dependent round trip below goes to HBM.
    {
        auto pf = [](const void *q) { asm volatile("prefetch.global.L2 [%0];" ::"l"(q)); };
        const int T = p.T;
        if (tid == 0) pf(p.plan);
        if (p.inkernel_route) {
            if (tid * 16 < T) { pf(p.off + tid * 16); pf(p.len + tid * 16); }
            if (tid * 128 < T) pf(p.elig + tid * 128);
            if (p.tau && tid * 32 < T) pf(p.tau + tid * 32);
        }
        if (tid * 32 < T) pf(plan_view(p.plan, T).done + tid * 32);
    }
    __syncthreads();
    // everything above touched shared memory only and overlapped the previous kernel on the stream (PDL)
    if (!p.chained) pdl_wait();
    if (p.next_chained) pdl_launch_dependents();
    if (tid == 0) trace_stamp(p, 6);
    const PlanView pv = plan_view(p.plan, p.T);
    PlanHeader *const hdr = (PlanHeader *)p.plan;
    int n_tiles = 0;
    bool layout_ok = true;

    // -----------------------------------------------------------------------------------------
    // Self-cleaning state and the first scheduling unit, in ONE atomic. hdr->sched = {clean token of this (T, W)
    // shape, next unit}: unit_cursor, finish_count, the per-tensor completion counters done[] and the exact
    // accumulators acc[] are all zero whenever the high half holds the token, because every call leaves them so
    // (slots are cleared by whoever rounds them, the grid's last CTA resets the rest and the low half). The
    // producer lane adds 1 here; the routing below needs none of that state and overlaps the round trip. A
    // returned value with the token in it is a valid unit of a clean plan. Anything else (first use of the
    // buffer, another shape) is settled once by compare-and-swap: the winning CTA zeroes the state and publishes
    // the token, the others wait for a CTA that is running. No grid-wide barrier, no cooperative launch: nothing
    // here assumes that all CTAs of the grid are resident together.
    // -----------------------------------------------------------------------------------------
    const uint32_t want_token = clean_token(p.T, W);
    const bool is_prod = (warp == kCW && lane == 0);
    unsigned long long sched_old = 0ull;
    if (p.inkernel_route && is_prod) sched_old = atomicAdd(&hdr->sched, 1ull);

    if (p.inkernel_route) {
        // ---- step a1 inside this kernel (T <= kMetaCap) --------
        // Every CTA derives the routing of the bucket into its shared-memory metadata (redundant O(T)
        // work, no dependence on another kernel or CTA); CTA 0 also writes the a1 outputs and the plan.
        const int T = p.T;
        PlanLayout PL = plan_layout(T);
        char *pb = (char *)p.plan;
        long long l = 0, o = 0, v_tiles = 0, v_words = 0, v_nl = 0;
        int r = NF_ROUTE_P;
        int bad = 0;
        if (tid < T) {
            if (!early_meta) {
                m_o = __ldg(p.off + tid);
                m_l = __ldg(p.len + tid);
                m_pe = tid == 0 ? 0 : __ldg(p.off + tid - 1) + __ldg(p.len + tid - 1);
                m_el = __ldg(p.elig + tid);
                if (p.tau) m_tau = __ldg(p.tau + tid);
            }
            o = m_o;
            l = m_l;
            const long long prev_end = m_pe;
            if (l < 0 || o < prev_end || o + l > p.n) bad = 1;
            if (l < 0) l = 0;
            if (!p.st.admitted) r = NF_ROUTE_P;
            else if (m_el == 0) r = NF_ROUTE_P;
            else if (p.st.veto || !p.st.capacity_ok) r = NF_ROUTE_F;
            else r = NF_ROUTE_L;
            v_tiles = (l + kTile - 1) / kTile;
            if (r == NF_ROUTE_L) { v_words = (l + 31) / 32; v_nl = 1; }
        }
        // exclusive scan of (tiles, words, nl) over the first kMetaCap threads (8 warps)
        long long i_tiles = v_tiles, i_words = v_words, i_nl = v_nl;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const long long a = __shfl_up_sync(0xffffffffu, i_tiles, d), b = __shfl_up_sync(0xffffffffu, i_words, d),
                            c = __shfl_up_sync(0xffffffffu, i_nl, d);
            if (lane >= d) { i_tiles += a; i_words += b; i_nl += c; }
        }
        if (tid == 0) trace_stamp(p, 9);
        long long *s_scan = reinterpret_cast<long long *>(smem_raw + 128);        // [3][8] warp totals, [24..27] tallies
        if (tid < 32) s_scan[tid] = 0;
        __syncthreads();
        if (warp < kMetaCap / 32 && lane == 31) { s_scan[warp] = i_tiles; s_scan[8 + warp] = i_words; s_scan[16 + warp] = i_nl; }
        if (blockIdx.x == 0 && warp < kMetaCap / 32) {
            // summary tallies (CTA 0 publishes them): warp sums by shuffle, one shared-memory add per warp
            // (64-bit shared-memory atomics are compare-and-swap loops: one per tensor cost 5 us at T = 96)
            unsigned long long *tal = reinterpret_cast<unsigned long long *>(s_scan + 24);
            const bool in = tid < T;
            unsigned q_f = (in && r == NF_ROUTE_F) ? 1u : 0u, q_p = (in && r == NF_ROUTE_P) ? 1u : 0u;
            long long e_l = (in && r == NF_ROUTE_L) ? l : 0, e_all = in ? l : 0;
            q_f = warp_sum(q_f);
            q_p = warp_sum(q_p);
#pragma unroll
            for (int d = 16; d >= 1; d >>= 1) {
                e_l += __shfl_xor_sync(0xffffffffu, e_l, d);
                e_all += __shfl_xor_sync(0xffffffffu, e_all, d);
            }
            if (lane == 0) {
                atomicAdd(tal + 0, (unsigned long long)q_f);
                atomicAdd(tal + 1, (unsigned long long)q_p);
                atomicAdd(tal + 2, (unsigned long long)e_l);
                atomicAdd(tal + 3, (unsigned long long)e_all);
            }
        }
        const int any_bad = __syncthreads_or(bad);
        if (tid == 0) trace_stamp(p, 10);
        long long b_tiles = 0, b_words = 0, b_nl = 0, t_tiles = 0, t_words = 0, t_nl = 0;
#pragma unroll
        for (int k = 0; k < kMetaCap / 32; ++k) {
            if (k < warp) { b_tiles += s_scan[k]; b_words += s_scan[8 + k]; b_nl += s_scan[16 + k]; }
            t_tiles += s_scan[k]; t_words += s_scan[8 + k]; t_nl += s_scan[16 + k];
        }
        const long long ex_tiles = b_tiles + i_tiles - v_tiles, ex_words = b_words + i_words - v_words,
                        ex_nl = b_nl + i_nl - v_nl;
        // (a plane row shorter than the packed words of the bucket would be overrun: refused like a bad layout)
        const int status = (any_bad || t_tiles > 0x3fffffffLL || (p.P && t_words > p.plane_stride)) ? NF_ERR_ARG : NF_OK;
        if (tid < T) {
            sm.m_tile[tid] = (int32_t)ex_tiles;
            sm.m_off[tid] = o;
            sm.m_len[tid] = l;
            sm.m_woff[tid] = r == NF_ROUTE_L ? ex_words : -1;
            sm.m_tau[tid] = (p.tau && r == NF_ROUTE_L) ? m_tau : 0.f;
        }
        if (tid == 0) sm.m_tile[T] = (int32_t)t_tiles;
        if (blockIdx.x == 0) {
            int32_t *tile_prefix = (int32_t *)(pb + PL.tile_prefix);
            int32_t *lt_index = (int32_t *)(pb + PL.lt_index);
            int64_t *lt_woff = (int64_t *)(pb + PL.lt_woff);
            LtRec *lt_rec = (LtRec *)(pb + PL.lt_rec);
            if (tid < T) {
                p.route_w[tid] = (uint8_t)r;
                p.woff_w[tid] = r == NF_ROUTE_L ? ex_words : -1;
                tile_prefix[tid] = (int32_t)ex_tiles;
                if (r == NF_ROUTE_L) {
                    lt_index[ex_nl] = tid;
                    lt_woff[ex_nl] = ex_words;
                    lt_rec[ex_nl] = LtRec{tid, o, l, ex_words, ex_words + v_words, 0};
                }
            }
            if (tid == 0) {
                const unsigned long long *tal = reinterpret_cast<const unsigned long long *>(s_scan + 24);
                tile_prefix[T] = (int32_t)t_tiles;
                lt_woff[t_nl] = t_words;
                hdr->magic = kPlanMagic;
                hdr->status = status;
                hdr->T = T;
                hdr->nL = (int32_t)t_nl;
                hdr->n = p.n;
                hdr->Wd = t_words;
                hdr->n_tiles = status == NF_OK ? (int32_t)t_tiles : 0;
                hdr->acc_slots = p.acc_slots;
                p.summary[NF_SUM_WD] = t_words;
                p.summary[NF_SUM_NL] = t_nl;
                p.summary[NF_SUM_NF] = (int64_t)tal[0];
                p.summary[NF_SUM_NP] = (int64_t)tal[1];
                p.summary[NF_SUM_E] = (int64_t)tal[2];
                p.summary[NF_SUM_F] = (int64_t)(tal[3] - tal[2]);
                p.summary[NF_SUM_TILES] = t_tiles;
                p.summary[NF_SUM_STATUS] = status;
            }
        }
        // a refused layout is a bucket without tiles: nothing is read or written, the plan's state (and the tail
        // of a previous bucket of the step) is still looked after
        layout_ok = status == NF_OK;
        n_tiles = layout_ok ? (int)t_tiles : 0;
        if (tid == 0) trace_stamp(p, 11);
    } else {
        if (pv.hdr->magic != kPlanMagic || pv.hdr->status != NF_OK) return;
        if (p.P && pv.hdr->Wd > p.plane_stride) {              // plane rows too short: refuse, like a bad layout
            if (blockIdx.x == 0 && tid == 0) { hdr->status = NF_ERR_ARG; p.summary[NF_SUM_STATUS] = NF_ERR_ARG; }
            return;
        }
        n_tiles = pv.hdr->n_tiles;
        if (is_prod) sched_old = atomicAdd(&hdr->sched, 1ull);
        if (p.T <= kMetaCap) {
            // per-tensor metadata -> shared memory (one round trip for the whole CTA)
            for (int t = tid; t <= p.T; t += kFThreads) {
                sm.m_tile[t] = __ldg(pv.tile_prefix + t);
                if (t < p.T) {
                    const bool isL = __ldg(p.route + t) == NF_ROUTE_L;
                    sm.m_off[t] = __ldg(p.off + t);
                    sm.m_len[t] = __ldg(p.len + t);
                    sm.m_woff[t] = isL ? __ldg(p.woff + t) : -1;
                    sm.m_tau[t] = (p.tau && isL) ? __ldg(p.tau + t) : 0.f;
                }
            }
        }
    }

    // ---- settle the clean token (the producer lane took a unit before the routing) -----------------
    if (is_prod) sm.flag[0] = ((uint32_t)(sched_old >> 32) == want_token) ? 0 : 1;
    __syncthreads();                                           // also: the shared-memory metadata is complete
    if (sm.flag[0]) {
        // rare: the plan's state is not known to be clean
        if (tid == 0) {
            int role = 0;                                      // 1: this CTA zeroes the state, 2: gave up
            for (unsigned spins = 0;; ++spins) {
                const unsigned long long v = ld_acquire_u64(&hdr->sched);
                const uint32_t hi = (uint32_t)(v >> 32);
                if (hi == want_token) break;
                if (hi == kInitToken) {
                    __nanosleep(200);
                    if (spins > (1u << 24)) { report_timeout(p); role = 2; break; }
                } else if (atomicCAS(&hdr->sched, v, (unsigned long long)kInitToken << 32) == v) {
                    role = 1;
                    break;
                }
            }
            sm.flag[1] = role;
        }
        __syncthreads();
        const int role = sm.flag[1];
        if (role == 2) return;
        if (role == 1) {
            const size_t na = (size_t)W * p.T * kAccWords;
            for (size_t i = tid; i < na; i += kFThreads) pv.acc[i] = 0ull;
            for (int t = tid; t < p.T; t += kFThreads) { pv.done[t] = 0; pv.fin[t] = 0ull; }
            for (int i = tid; i < kMaxOrphans; i += kFThreads) pv.orph[i] = 0;
            if (tid == 0) { hdr->unit_cursor = 0; hdr->finish_count = 0; }
            __threadfence();
            __syncthreads();
            if (tid == 0) atomicExch(&hdr->sched, (unsigned long long)want_token << 32);
        }
        __syncthreads();
        if (is_prod) {
            sched_old = atomicAdd(&hdr->sched, 1ull);
            if ((uint32_t)(sched_old >> 32) != want_token) { report_timeout(p); sched_old = 0x7fffffffull; }
        }
    }
    if (tid == 0) trace_stamp(p, 7);

    const DecodeSrc own{p.T, n_tiles, p.T <= kMetaCap, pv.tile_prefix, p.off, p.len, p.woff, p.route, pv.fin, p.dirs, p.out, hdr, pv.orph};
    const PlanView ppv = plan_view(p.prev_plan, p.prev_T);              // (only dereferenced when chained)
    DecodeSrc prev{p.prev_T, 0, false, ppv.tile_prefix, p.prev_off, p.prev_len, p.prev_woff, p.prev_route, ppv.fin, p.prev_dirs,
                   p.prev_out, (PlanHeader *)p.prev_plan, ppv.orph};

    // scheduling units: a pure function of (n_tiles, grid): 4 consecutive tiles, then 2, then single tiles near
    // the end (guided self-scheduling with fixed boundaries). A *segment* = unit x tensor is what one FP32
    // partial spans, so the value of every partial depends on the data only, not on which CTA took the unit.
    const int sA = max(0, n_tiles - (MULTI ? NF_TAIL4_M : NF_TAIL4) * (int)gridDim.x) & ~3, nA = sA >> 2;
    const int sB = sA + (max(0, n_tiles - (MULTI ? NF_TAIL2_M : NF_TAIL2) * (int)gridDim.x - sA) & ~1), nB = (sB - sA) >> 1;

    if (warp == kCW) {
        // =====================================================================================
        // producer (one elected lane): issues the bulk copies of every (tile, worker group) of the units it
        // takes from the device-wide cursor; a CTA that runs ahead (SM position, co-running decode warps)
        // simply takes more. The stage carries its tile index (and whether the tile ends a segment).
        // =====================================================================================
        if (lane == 0) {
            const uint64_t pol = policy_evict_first();
            // Units are taken several at a time while plenty are left (guided: a share of what remains when the
            // previous trip was made, 1 .. NF_GRAB): fewer trips to one address, and a CTA walks longer contiguous
            // stretches of the W rows (DRAM pages, TLB entries). The segment boundaries are those of the units, so
            // how many are taken at once changes nothing in the values.
            int u_next = (int)(uint32_t)sched_old;                 // the unit taken before the routing
            int u_end = u_next + 1;
            // Deferred tail: this bucket's state stays in use after the kernel, so the clean token must go (a call that
            // found it would take the state for clean). It may go once no CTA of this grid will look at it again, i.e.
            // when every CTA has made its first draw: finish_count counts the CTAs that have (this one's draw has
            // returned: its token was checked above); the last one to start takes the token away when it leaves.
            int started = -1;
            if (p.defer_tail) started = atomicAdd(&hdr->finish_count, 1);
            const int n_units = nA + nB + (n_tiles - sB);
            int pr_st = 0, pr_next = 0, pr_end = 0;
            uint32_t pr_ph = 0;
            TensorCur pc{};
            pc.tile_e = 0;
            for (;;) {
                if (pr_next >= pr_end) {
                    if (u_next >= u_end) {
                        const int g = min(max((n_units - u_end) / (4 * (int)gridDim.x), 1), NF_GRAB);
                        u_next = (int)(uint32_t)atomicAdd(&hdr->sched, (unsigned long long)g);
                        u_end = u_next + g;
                    }
                    const int u = u_next++;
                    if (u < nA) { pr_next = 4 * u; pr_end = pr_next + 4; }
                    else if (u < nA + nB) { pr_next = sA + 2 * (u - nA); pr_end = pr_next + 2; }
                    else { pr_next = sB + (u - nA - nB); pr_end = pr_next + 1; }
                }
                const int pr_tile = pr_next;
                if (pr_tile >= n_tiles) {
                    mbar_wait(sm.empty + pr_st, pr_ph ^ 1u);
                    sm.tile_of[pr_st] = -1;                            // sentinel: the consumers stop
                    mbar_arrive(sm.full + pr_st);
                    // deferred tail: the CTA's decode warps wind down now (they need a few us to finish the span they
                    // are storing and to hand on what else they hold), while the consumers work off the ring
                    if (p.defer_tail) *(volatile int *)(sm.flag + 4) = 1;
                    if (started == (int)gridDim.x - 1) {
                        hdr->finish_count = 0;
                        atomicAnd(&hdr->sched, 0xffffffffull);         // not clean until the next kernel has drained the tail
                    }
                    break;
                }
                if (pr_tile >= pc.tile_e) tensor_lookup(p, pv, sm, pr_tile, pc);
                // run = the tiles of this unit inside the current tensor (one segment). Several worker groups
                // (MULTI), low-bit or health: its stages go group-major (group 0 of tiles 0..R-1, then group 1,
                // ...), so that the consumers flush the FP32 partials of a group once per run.
                // (FP32-route tiles carry one running FP32 sum across the groups: they go one tile at a time.)
                const int seg_len = min(pr_end, pc.tile_e) - pr_tile;   // <= 4
                const int R = (MULTI && pc.isL) ? seg_len : 1;
                pr_next += R;
                for (int w0 = 0; w0 < (MULTI ? W : 1); w0 += kGroup) {
                    const int nw = MULTI ? min(kGroup, W - w0) : W;
                    for (int r = 0; r < R; ++r) {
                        const int64_t tile_base = (int64_t)(pr_tile + r - pc.tile_b) * kTile;
                        const int64_t rem = pc.len - tile_base;
                        const int need = rem >= kTile ? kTile : (int)rem;
                        // aligned rows: whole float4s only (a partial one is read from global memory by its owner
                        // thread). Unaligned rows: from the 16-byte boundary below the row to the one above its end
                        // (whole 16-byte chunks, each holding at least one element of the row).
                        const uint32_t bytes = (uint32_t)((need & ~3) * 4);
                        const float *src = p.g + pc.off + tile_base;
                        const int st = pr_st;
                        mbar_wait(sm.empty + st, pr_ph ^ 1u);                  // first lap: passes at once
                        sm.tile_of[st] = pr_tile + r;
                        sm.seg_of[st] = MULTI ? 1 : (seg_len == 1);
                        if (MULTI) sm.run_of[st] = R;
                        float *dst = sm.ring + (size_t)st * kStageFloats;
                        if (!pc.aligned) {
                            uint32_t tx = 0;
                            for (int w = 0; w < nw; ++w)
                                tx += (uint32_t)((((int)((pc.off + (int64_t)(w0 + w) * p.worker_stride) & 3) + need + 3) & ~3) * 4);
                            mbar_expect_tx(sm.full + st, tx);
                            for (int w = 0; w < nw; ++w) {
                                const int m = (int)((pc.off + (int64_t)(w0 + w) * p.worker_stride) & 3);
                                bulk_g2s(dst + w * kPitch, src + (size_t)(w0 + w) * p.worker_stride - m,
                                         (uint32_t)(((m + need + 3) & ~3) * 4), sm.full + st, pol);
                            }
                        } else if (bytes) {
                            mbar_expect_tx(sm.full + st, (uint32_t)nw * bytes);
                            for (int w = 0; w < nw; ++w)
                                bulk_g2s(dst + w * kPitch, src + (size_t)(w0 + w) * p.worker_stride, bytes, sm.full + st, pol);
                        } else {
                            mbar_arrive(sm.full + st);
                        }
                        if (++pr_st == stages) { pr_st = 0; pr_ph ^= 1u; }
                    }
                }
            }
        }
    } else if (warp == kCW + 1) {
        // =====================================================================================
        // housekeeping warp: the outputs nobody else writes. Tensors that own no tile (len = 0): totals 0, scale 0 on
        // the FP32 route and the oracle's 0/0 on the low-bit route. FP32-route tensors: scale 0, and abs_sum 0 when no
        // health statistics are gathered (with them, the tensor is finalised like any other by its last arriver).
        // =====================================================================================
        for (int t = blockIdx.x * 32 + lane; t < p.T && layout_ok; t += (int)gridDim.x * 32) {
            int64_t len_t;
            bool isL;
            if (p.T <= kMetaCap) { len_t = sm.m_len[t]; isL = sm.m_woff[t] >= 0; }
            else { len_t = __ldg(p.len + t); isL = __ldg(p.route + t) == NF_ROUTE_L; }
            if (len_t > 0 && isL) continue;
            if (len_t <= 0 || !HEALTH) {
                for (int w = 0; w < W; ++w) {
                    const size_t o = (size_t)w * p.T + t;
                    p.abs_sum[o] = 0.0;
                    if (HEALTH) { p.sumsq[o] = 0.0; p.nan_cnt[o] = 0ull; p.inf_cnt[o] = 0ull; }
                }
            }
            double s = 0.0;
            const double zero = 0.0, dl = (double)len_t;
            for (int w = 0; w < W; ++w) s += (double)(float)(zero / dl);
            const float S = isL ? (float)(s / (double)W) : 0.f;
            pv.scale[t] = S;
            if (p.scale_out) p.scale_out[t] = S;
        }
        // ---- then the CTA's reducer and publisher. The 16 consumer warps hand it records through two buffers: a warp
        // arrives on the buffer's named barrier and goes on (it waits on the buffer's "free"
        // mbarrier only when it comes back to the same buffer), so the consumers never wait for each other here.
        //  * data record = a SEGMENT (the tiles of one scheduling unit inside one tensor), at most kRecW workers of it
        //    (wider fan-in: several records per segment): 16 FP64 values per (worker,
        //    statistic), one per consumer warp; a lane per (worker, statistic) sums them in warp order (a fixed shape:
        //    the value depends on the data only) and adds the segment's total EXACTLY to the tensor's accumulator
        //    (integer atomics: the order in which segments arrive, i.e. the dynamic scheduling, cannot change the
        //    result); the NaN / Inf tallies of the segment go the same way.
        //  * flush record = this CTA is through with tensor t for now (`n` tiles since its last flush): publish the
        //    count (release: every consumer warp arrived after its last store of the tensor; this warp's fence is
        //    cumulative) and, if that completed the tensor, finalise it (finalize_tensor_warp).
        {
            const int T = p.T, Wc = fused_recw(W);
            int b = 0;
            for (;;) {
                seg_bar_sync(b);
                const int *rec = sm.seg_rec + 8 * b;
                const int t = rec[0];
                if (t < 0) break;
                const bool isL = rec[2] != 0;
                const int wbase = rec[5], wc = min(Wc, W - wbase);     // data records: the workers the record covers
                if (rec[1] == 2) {
                    // the segment is the whole tensor: its sums ARE the totals (exactly what rounding the accumulator
                    // of a single addend gives)
                    const int64_t len_t = *reinterpret_cast<const int64_t *>(rec + 6);
                    const double *src0 = sm.wacc + (size_t)b * kCW * 2 * Wc;
                    for (int j0 = 0; j0 < 2 * wc; j0 += 32) {
                        const int j = j0 + lane, wr = j >> 1, w = wbase + wr;
                        double tot = 0.0;
                        if (j < 2 * wc) {
#pragma unroll
                            for (int k = 0; k < kCW; ++k) tot += src0[(size_t)k * 2 * Wc + j];
                        }
                        const double other = __shfl_xor_sync(0xffffffffu, tot, 1);      // even lane: sum |x|, odd lane: sum x^2
                        if (j < 2 * wc && (j & 1) == 0) {
                            const unsigned cn_ = atomicExch(&sm.nan[b * 32 + wr], 0u), ci_ = atomicExch(&sm.inf[b * 32 + wr], 0u);
                            const size_t o = (size_t)w * T + t;
                            double A = 0.0;
                            if (isL) {
                                A = tot;
                                if (cn_) A = __longlong_as_double(0x7ff8000000000000ll);
                                else if (ci_) A = __longlong_as_double(0x7ff0000000000000ll);
                            }
                            p.abs_sum[o] = A;
                            if (HEALTH) { p.sumsq[o] = other; p.nan_cnt[o] = cn_; p.inf_cnt[o] = ci_; }
                            sm.sw[w] = (float)(A / (double)len_t);
                        }
                    }
                    __syncwarp();
                    if (isL && lane == 0 && wbase + wc == W) {             // the tensor's last record: all W scales are in
                        double sacc = 0.0;
                        for (int w = 0; w < W; ++w) sacc += (double)sm.sw[w];
                        const float S = (float)(sacc / (double)W);
                        pv.scale[t] = S;
                        if (p.scale_out) p.scale_out[t] = S;
                        st_release_u64(pv.fin + t, (1ull << 32) | (unsigned long long)__float_as_uint(S));
                    }
                } else if (rec[1] == 0) {
                    const double *src0 = sm.wacc + (size_t)b * kCW * 2 * Wc;
                    for (int j = lane; j < 2 * wc; j += 32) {
                        const double *src = src0 + j;
                        double tot = 0.0;
#pragma unroll
                        for (int k = 0; k < kCW; ++k) tot += src[(size_t)k * 2 * Wc];
                        unsigned long long *slot = pv.acc + ((size_t)(wbase + (j >> 1)) * T + t) * kAccWords;
                        if ((j & 1) == 0) { if (isL) acc_add(slot + kAccAbs, kAccAbsWords, kAccAbsBase, tot); }
                        else if (HEALTH) acc_add(slot + kAccSq, kAccSqWords, kAccSqBase, tot);
                    }
                    for (int w = lane; w < wc; w += 32) {
                        const unsigned cn_ = atomicExch(&sm.nan[b * 32 + w], 0u), ci_ = atomicExch(&sm.inf[b * 32 + w], 0u);
                        unsigned long long *slot = pv.acc + ((size_t)(wbase + w) * T + t) * kAccWords;
                        if (cn_) atomicAdd(slot + kAccNan, (unsigned long long)cn_);
                        if (ci_) atomicAdd(slot + kAccInf, (unsigned long long)ci_);
                    }
                } else {
                    const int n = rec[3], total = rec[4];
                    const int64_t len_t = *reinterpret_cast<const int64_t *>(rec + 6);
                    __threadfence();
                    __syncwarp();
                    int old = 0;
                    if (lane == 0) old = atomicAdd(pv.done + t, n);
                    old = __shfl_sync(0xffffffffu, old, 0);
                    if (old + n == total) {
                        // (every other CTA's adds of the tensor were fenced before its own count reached done[t]; the
                        // slots are read from L2, after the value the atomic returned: control dependency)
                        if (lane == 0) trace_stamp(p, 12);
                        finalize_tensor_warp<HEALTH>(p, pv, sm, t, len_t, isL, lane);
                        if (lane == 0) trace_stamp(p, 13);
                    }
                }
                __syncwarp();
                if (lane == 0) mbar_arrive(sm.seg_free + b);   // (release: what was done is ordered before whoever waits)
                b ^= 1;
            }
        }
    } else if (warp >= kCW + 2) {
        // =====================================================================================
        // decode warps (pass B inside the kernel): see decode_warp_loop(). The consumers join them once
        // their own tiles are done.
        // =====================================================================================
        // Chaining: the decode of a bucket's LAST low-bit tensor cannot start before the bucket has been read
        // completely (S_t needs all of the tensor), so at the end of a stand-alone call the device only writes. Inside
        // a step the kernels of consecutive buckets form a pipeline instead: when pass A of bucket k ends, its CTAs
        // leave at once (defer_tail) and the kernel of bucket k+1, which needs nothing of bucket k for its own
        // pass A and therefore never waited for it, drains bucket k's remaining units here, beside its own reads.
        // The only thread-level dependency waits of a chained kernel are the ones in front of bucket k's data.
        const int dwarp = warp - (kCW + 2);
        if (p.chained) {
            pdl_wait();
            prev.n_tiles = __ldcg(&prev.hdr->n_tiles);
            if (lane == 0) sm.aux[0] = prev.n_tiles + 1;
            // the bucket before the previous one: kernel k-1 is complete, and it had waited for kernel k-2
            if (p.pp_plan && blockIdx.x == 0 && dwarp == 0) reset_bucket_state(p.pp_plan, p.pp_T, p.pp_W, lane);
            {
                // first the units the previous kernel's decode warps had in hand when their CTAs left (all final by
                // now): this warp takes, and clears, the entries of the same warp of CTAs c, c + grid, ...
                DecodeCur dc{-1, 0, 0, 0, 0, 0, false, 0.f};
                for (int c = (int)blockIdx.x; (c * kDW + dwarp + 1) * kHandOn <= kMaxOrphans; c += (int)gridDim.x) {
                    int4 *e = reinterpret_cast<int4 *>(prev.orph + (c * kDW + dwarp) * kHandOn);
                    const int4 v = __ldcg(e);
                    if ((v.x | v.y | v.z | v.w) == 0) continue;
                    if (lane == 0) __stcg(e, make_int4(0, 0, 0, 0));
                    if (v.x) decode_span(p, prev, sm, dc, v.x - 1, v.x, lane);
                    if (v.y) decode_span(p, prev, sm, dc, v.y - 1, v.y, lane);
                    if (v.z) decode_span(p, prev, sm, dc, v.z - 1, v.z, lane);
                    if (v.w) decode_span(p, prev, sm, dc, v.w - 1, v.w, lane);
                }
            }
            if (p.next_chained) {
                // middle of a chain: the warp leaves the previous bucket when this CTA's pass A is about to end (what
                // is left then, the consumers take, see there); flag[5] = some decode warp saw the cursor exhausted
                const bool exhausted = decode_warp_loop(p, prev, sm, sm.flag + 4, false, nullptr, lane, dwarp);
                if (exhausted && lane == 0) *(volatile int *)(sm.flag + 5) = 1;
            } else {
                decode_warp_loop(p, prev, sm, nullptr, false, nullptr, lane, dwarp);
                through_with_prev(p, prev.hdr, ppv, sm, lane);
            }
        }
        decode_warp_loop(p, own, sm, p.defer_tail ? sm.flag + 4 : nullptr, true, sm.flag + 7, lane, dwarp);
        if (warp == kCW + 2 && lane == 0) trace_stamp(p, 4);
    } else {
        // =====================================================================================
        // consumers
        // =====================================================================================
        const int ctid = tid;                       // 0..511
        if (ctid == 0) trace_stamp(p, 0);
        const TCtl tctl = make_tctl(lane);
        const bool ternary = p.ternary != 0;
        float af[8], qf[8];                         // FP32 partials of the current worker group
#pragma unroll
        for (int i = 0; i < 8; ++i) { af[i] = 0.f; qf[i] = 0.f; }
        int kcnt = 0;
        int4 recent = make_int4(0, 0, 0, 0);        // the last tiles accumulated in af/qf, most recent first
        int st = 0;
        uint32_t ph = 0;
        TensorCur c{};
        c.tile_e = 0;
        c.t = -1;
        bool touched = false;                       // this CTA processed tiles of tensor c.t
        int ntile_acc = 0;                          // tiles of tensor c.t this CTA has finished
        uint32_t *pP = nullptr, *pN = nullptr;      // this thread's plane-word / direction / output slots
        uint8_t *pD = nullptr;                      //   of tile 0 of the current tensor
        float *pO = nullptr;
        int segpar = 0;                             // buffer of the current record's per-warp FP64 values
        double *wbuf = sm.wacc;

        uint32_t seguse0 = 0u, seguse1 = 0u;        // uses of each segment buffer so far
        // before the first stat_flush of a segment: the reducer warp is through with the buffer's previous segment
        auto seg_acquire = [&]() __attribute__((always_inline)) {
            const uint32_t u = segpar ? seguse1 : seguse0;
            mbar_wait_backoff(sm.seg_free + segpar, (u & 1u) ^ 1u);    // first use: passes at once
        };
        // after the last stat_flush of a segment: hand the buffer to the reducer warp (see there) and go on
        auto seg_publish = [&](int t, int kind, bool isL, int n, int total, int64_t len_t, int wbase) __attribute__((always_inline)) {
            if (ctid == 0) {
                int *rec = sm.seg_rec + 8 * segpar;
                rec[0] = t; rec[1] = kind; rec[2] = isL ? 1 : 0; rec[3] = n; rec[4] = total; rec[5] = wbase;
                *reinterpret_cast<int64_t *>(rec + 6) = len_t;
            }
            seg_bar_arrive(segpar);
            if (segpar) ++seguse1; else ++seguse0;
            segpar ^= 1;
            wbuf = sm.wacc + (size_t)segpar * kCW * 2 * fused_recw(W);
        };
        // All tiles this CTA took of tensor c.t so far are done: tell the reducer warp (a flush record: it publishes the
        // tile count and finalises the tensor if that completed it). No barrier, no round trip on the consumers' path:
        // every warp arrives after its own last store of the tensor.
        auto flush_tensor = [&]() __attribute__((always_inline)) {
            if (c.isL || HEALTH) {
                seg_acquire();
                seg_publish(c.t, 1, c.isL, ntile_acc, c.tile_e - c.tile_b, c.len, 0);
            }
            ntile_acc = 0;
        };

        for (;;) {
            mbar_wait(sm.full + st, ph);
            const int tile = sm.tile_of[st];
            if (tile < 0) break;
            if (tile >= c.tile_e) {
                if (touched) flush_tensor();
                tensor_lookup(p, pv, sm, tile, c);
                touched = false;
                const size_t pl = (size_t)(lane & 7) * p.plane_stride + c.woff + warp * 4 + (lane >> 3);
                pP = (c.isL && p.P) ? p.P + pl : nullptr;
                pN = (c.isL && p.P && ternary) ? p.N + pl : nullptr;
                pD = c.isL ? p.dirs + (size_t)c.woff * 8 + ctid : nullptr;
                pO = p.out + c.off + 4 * ctid;
            }
            const int rel = tile - c.tile_b;
            const bool stats = c.isL || HEALTH;     // this tensor's totals are wanted
            // MULTI: the producer sends a run of R consecutive tiles (one segment) group-major (see there)
            const int R = MULTI ? sm.run_of[st] : 1;
            const bool seg_end = MULTI ? true : (sm.seg_of[st] != 0);
            if (MULTI) recent = make_int4(tile + R - 1, tile + R - 2, tile + R - 3, tile + R - 4);
            else recent = make_int4(tile, recent.x, recent.y, recent.z);
            uint32_t posR = 0u, negR = 0u;
            uint32_t cp0 = 0u, cp1 = 0u, cp2 = 0u, cp3 = 0u;     // byte-packed running counts of the run's tiles (MULTI)
            uint32_t cn0 = 0u, cn1 = 0u, cn2 = 0u, cn3 = 0u;
            float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
            int valid = 0;
            for (int w0 = 0; w0 < (MULTI ? W : 1); w0 += kGroup) {   // one ring stage per (tile, worker group)
                const int nw = MULTI ? min(kGroup, W - w0) : W;
                for (int r = 0; r < R; ++r) {
                    if (MULTI && (w0 > 0 || r > 0)) mbar_wait(sm.full + st, ph);
                    const float *sb = sm.ring + (size_t)st * kStageFloats + 4 * ctid;
                    uint64_t *const empty_bar = sm.empty + st;
                    if (++st == stages) { st = 0; ph ^= 1u; }
                    const int64_t rem_t = c.len - (int64_t)(rel + r) * kTile;
                    const bool ragged = rem_t < kTile;              // last tile of the tensor, need < kTile elements
                    const int need = ragged ? (int)rem_t : kTile;
                    valid = min(max(need - 4 * ctid, 0), 4);
                    if (MULTI) { posR = 0u; negR = 0u; }
                    if (ragged || !c.aligned) {
                        slow_tile<HEALTH>(sb, p.g + (size_t)w0 * p.worker_stride + c.off + (int64_t)(rel + r) * kTile + 4 * ctid,
                                          p.worker_stride, nw, valid, !c.aligned, (int)((c.off + (int64_t)w0 * p.worker_stride) & 3),
                                          (int)(p.worker_stride & 3), c.isL, ternary, c.tau, -c.tau, af, qf, posR, negR, acc,
                                          w0 == 0);
                    } else if (c.isL) {
                        const float tau = c.tau, ntau = -c.tau;
                        if (ternary) {
                            if (nw == kGroup) fast_signs<2, HEALTH, true>(sb, nw, tau, ntau, af, qf, posR, negR);
                            else fast_signs<2, HEALTH, false>(sb, nw, tau, ntau, af, qf, posR, negR);
                        } else {
                            if (nw == kGroup) fast_signs<1, HEALTH, true>(sb, nw, tau, ntau, af, qf, posR, negR);
                            else fast_signs<1, HEALTH, false>(sb, nw, tau, ntau, af, qf, posR, negR);
                        }
                    } else {
                        acc = (nw == kGroup) ? fast_fp32<HEALTH, true>(sb, nw, af, qf, acc, w0 == 0)
                                             : fast_fp32<HEALTH, false>(sb, nw, af, qf, acc, w0 == 0);
                    }
                    __syncwarp();
                    if (lane == 0) mbar_arrive(empty_bar);          // every lane's reads of the stage are done
                    if (c.isL) {
                        if (pP) {
                            // packed plane words: 8x8 nibble transpose, lane q of an octet stores worker q's word
                            const bool stp = ((lane & 7) < nw) && (32 * (warp * 4 + (lane >> 3)) < need);
                            const size_t o = (size_t)(rel + r) * (kTile / 32) + (size_t)w0 * p.plane_stride;
                            const uint32_t pw = nib_transpose8(posR, tctl);
                            if (stp) pP[o] = pw;
                            if (ternary) {
                                const uint32_t nwd = nib_transpose8(negR, tctl);
                                if (stp) pN[o] = nwd;
                            }
                        }
                        if (MULTI) {
                            uint32_t dp = 0u, dn = 0u;
#pragma unroll
                            for (int j = 0; j < 4; ++j) {
                                dp += (uint32_t)__popc(posR & (0x11111111u << j)) << (8 * j);
                                if (ternary) dn += (uint32_t)__popc(negR & (0x11111111u << j)) << (8 * j);
                            }
                            cp0 += r == 0 ? dp : 0u; cp1 += r == 1 ? dp : 0u; cp2 += r == 2 ? dp : 0u; cp3 += r == 3 ? dp : 0u;
                            cn0 += r == 0 ? dn : 0u; cn1 += r == 1 ? dn : 0u; cn2 += r == 2 ? dn : 0u; cn3 += r == 3 ? dn : 0u;
                        }
                    }
                }
                if (MULTI && stats) {
                    // a segment goes to the reducer warp in records of at most kRecW workers (the last one after the
                    // votes below)
                    if (w0 % kRecW == 0) seg_acquire();
                    stat_flush<HEALTH>(p, sm, wbuf, segpar * 32, af, qf, c.off, c.len, c.tile_b, w0, nw, R, recent, ctid, c.aligned);
                    if ((w0 + kGroup) % kRecW == 0 && w0 + kGroup < W)
                        seg_publish(c.t, R == c.tile_e - c.tile_b ? 2 : 0, c.isL, 0, 0, c.len, w0 + kGroup - kRecW);
                }
            }
            if (c.isL) {
                // majority vote with margin m and ties -> 0 (readings #3, #5, #6)
                if (!MULTI) {
                    const uint32_t d = ternary ? vote4<true>(posR, negR, W, p.margin) : vote4<false>(posR, negR, W, p.margin);
                    if (valid > 0) pD[(size_t)rel * (kTile / 4)] = (uint8_t)d;
                } else {
#pragma unroll
                    for (int r = 0; r < kKTiles; ++r) {
                        if (r < R) {
                            const uint32_t d = vote4_packed(r == 0 ? cp0 : (r == 1 ? cp1 : (r == 2 ? cp2 : cp3)),
                                                            r == 0 ? cn0 : (r == 1 ? cn1 : (r == 2 ? cn2 : cn3)), ternary, W, p.margin);
                            if (c.len - (int64_t)(rel + r) * kTile > 4 * ctid) pD[(size_t)(rel + r) * (kTile / 4)] = (uint8_t)d;
                        }
                    }
                }
            } else {
                float *o = pO + (size_t)rel * kTile;
                float4 r = acc;
                r.x = __fmul_rn(p.alpha, r.x); r.y = __fmul_rn(p.alpha, r.y);
                r.z = __fmul_rn(p.alpha, r.z); r.w = __fmul_rn(p.alpha, r.w);
                if (valid == 4 && c.aligned) {
                    __stcs(reinterpret_cast<float4 *>(o), r);
                } else {
                    if (valid > 0) o[0] = r.x;
                    if (valid > 1) o[1] = r.y;
                    if (valid > 2) o[2] = r.z;
                    if (valid > 3) o[3] = r.w;
                }
            }
            touched = true;
            ntile_acc += R;
            if (!MULTI) ++kcnt;
            if (stats && seg_end) {
                // a segment that IS the whole tensor (small tensors: norms, biases): this CTA is its only arriver, so
                // the reducer warp writes the tensor's results straight from the segment's sums (record kind 2): no
                // accumulator, no fence, no completion count, no flush record
                const bool whole = (MULTI ? R : kcnt) == c.tile_e - c.tile_b;
                if (!MULTI) {
                    seg_acquire();
                    stat_flush<HEALTH>(p, sm, wbuf, segpar * 32, af, qf, c.off, c.len, c.tile_b, 0, W, kcnt, recent, ctid, c.aligned);
                    kcnt = 0;
                }
                seg_publish(c.t, whole ? 2 : 0, c.isL, 0, 0, c.len, MULTI ? (W - 1) / kRecW * kRecW : 0);
                if (whole) { touched = false; ntile_acc = 0; }
            } else if (!MULTI && seg_end) {
                kcnt = 0;
            }
        }
        if (ctid == 0) trace_stamp(p, 1);
        if (touched && (c.isL || HEALTH) && p.next_chained) {
            // middle of a chain: the last tensor goes to the reducer warp like any other (its fence and its atomic are
            // two round trips: they overlap what the consumers do next, the previous bucket's backlog; the tensor's
            // decode is the next kernel's business anyway)
            flush_tensor();
        } else if (touched && (c.isL || HEALTH)) {
            // the last tensor this CTA worked on: its decode is now the critical path and the consumers are free, so
            // they publish and finalise it themselves (16 warps) once the reducer warp is through with every record
            if (seguse0 > 0u) mbar_wait_backoff(sm.seg_free + 0, (seguse0 - 1u) & 1u);
            if (seguse1 > 0u) mbar_wait_backoff(sm.seg_free + 1, (seguse1 - 1u) & 1u);
            consumer_sync();
            if (ctid == 0) {
                __threadfence();
                const int old = atomicAdd(pv.done + c.t, ntile_acc);
                sm.flag[1] = (old + ntile_acc == c.tile_e - c.tile_b) ? 1 : 0;
            }
            consumer_sync();
            if (sm.flag[1]) finalize_tensor<HEALTH>(p, pv, sm, c.t, c.len, c.isL, ctid);
        }
        seg_acquire();
        seg_publish(-1, 0, false, 0, 0, 0, 0);      // no more records: the reducer warp leaves
        if (ctid == 0) trace_stamp(p, 2);
        if (p.defer_tail && ctid == 0) *(volatile int *)(sm.flag + 4) = 1;   // this CTA's decode warps take no more units
        if (p.chained) {
            // The previous bucket's tail. If no decode warp of this CTA has seen its cursor exhausted there is a backlog
            // (the decode warps alone do not keep up with a bucket's worth of decoding per kernel): the consumers take
            // a share with all 16 warps. In the middle of a chain nothing is counted (see through_with_prev); the last
            // kernel of a chain counts its CTAs: there the consumers register as a third party before they help.
            if (ctid == 0)
                sm.flag[2] = p.next_chained ? (*(volatile int *)(sm.flag + 5) == 0 ? 1 : 0)
                                            : ((atomicCAS(sm.flag + 5, 0, 0x100) == 0) ? 1 : 0);
            consumer_sync();
            if (sm.flag[2]) {
                pdl_wait();
                const int seen = *(volatile int *)sm.aux;           // (read by the decode warps long ago)
                prev.n_tiles = seen ? seen - 1 : __ldcg(&prev.hdr->n_tiles);
                decode_cta_loop(p, prev, sm, ctid, 0);
                if (!p.next_chained && warp == 0) through_with_prev(p, prev.hdr, ppv, sm, lane);
            }
        }
        if (!p.defer_tail) decode_cta_loop(p, own, sm, ctid, *(volatile int *)(sm.flag + 7));      // help finish pass B
        if (ctid == 0) trace_stamp(p, 3);
    }

    // ---- the self-cleaning state at the end of the kernel. Tail not deferred (a stand-alone call, the last bucket of a
    // step): the grid's last CTA resets this bucket's state. Tail deferred: nothing to do here (the next kernel of the
    // step resets it when it is through with the tail; the last CTA to START took the clean token away, see the
    // producer), so such a CTA leaves without a device-wide round trip. The previous bucket's state was reset by the
    // decode warps. ----
    if (!p.defer_tail) {
        __syncthreads();
        if (tid == 0) {
            // (this CTA's stores to the state, the fin words of the tensors it finalised, must come first)
            __threadfence();
            const int old = atomicAdd(&hdr->finish_count, 1);
            const int last = (old == (int)gridDim.x - 1) ? 1 : 0;
            if (last) __threadfence();
            sm.flag[2] = last;
        }
        __syncthreads();
        if (sm.flag[2]) {
            for (int t = tid; t < p.T; t += kFThreads) { pv.done[t] = 0; pv.fin[t] = 0ull; }
            if (tid == 0) {
                hdr->finish_count = 0;
                hdr->unit_cursor = 0;
                hdr->sched = (unsigned long long)want_token << 32;
            }
        }
    }
    if (tid == 0) trace_stamp(p, 8);
}

// ---------------------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------------------
template <bool HEALTH, bool MULTI>
static cudaError_t launch_fused_t(const StreamParams &p, int64_t n, cudaStream_t s) {
    const int stages = kStages;                              // (the record buffers are at most 16 KB at any fan-in)
    const size_t smem = fused_smem_bytes(stages, p.W);
    static bool configured = false;
    if (!configured) {
        const size_t mx = fused_smem_bytes(kStages, kRecW);
        cudaError_t e = cudaFuncSetAttribute(fused_passA_kernel<HEALTH, MULTI>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                             (int)mx);
        if (e != cudaSuccess) return e;
        configured = true;
    }
    int64_t work = n / kTile + p.T;                          // upper bound of the tile count
    if (work <= 0) return cudaSuccess;
    int64_t grid = device_sm_count();                        // persistent: one CTA per SM
    if (grid > work) grid = work;
    // No cooperative launch: no CTA ever waits for a CTA that has not started, so the grid need
    // not be co-resident (other kernels may hold SMs, two calls may share the device).
    cudaError_t e = launch_kernel(fused_passA_kernel<HEALTH, MULTI>, (unsigned)grid, kFThreads, smem, s, true, p, stages);
    if (e != cudaSuccess) return e;
    return cudaGetLastError();
}

// The whole of pass A and pass B for one bucket: any W, any tensor offsets.
cudaError_t launch_fused_passA(bool health, const StreamParams &p, int64_t n, cudaStream_t s) {
    if (p.W > kGroup) return health ? launch_fused_t<true, true>(p, n, s) : launch_fused_t<false, true>(p, n, s);
    return health ? launch_fused_t<true, false>(p, n, s) : launch_fused_t<false, false>(p, n, s);
}

}  // namespace nf
