// nf_reduce.cu — step a3 (reducer-side compact sign-count aggregation + decode) and the two levels of
// the hierarchical count (NEXT-1). PAPER §5.2 L211 ("sum these
// indicators across workers ... majority voting ... writes the scaled aggregate direction back"),
// §6.1 L247 ("recovering per-coordinate sign counts rather than numerically adding packed
// machine words"), L76 (endpoint service = counting compact updates under fan-in W).
//
// a3 is a positional popcount over the W packed words of each word position. One thread owns one
// word position (32 elements): it streams the W words (coalesced across the warp, 8 independent
// loads in flight) through a bit-sliced carry-save adder tree (Harley-Seal style: 7 full adders
// per 8 words, ~3 LOP3 per word), which leaves the per-element counts as 8 bit-planes; the
// majority test with margin is then a bit-sliced compare that decides 32 elements at once.
// The FP32 output is written warp-cooperatively (lane = element) so stores are 128-byte coalesced.
#include "nf_internal.cuh"

namespace nf {

constexpr int kRThreads = 256;

// full adder on 32 bit-lanes: 2 LOP3
__device__ __forceinline__ void csa(uint32_t &carry, uint32_t &sum, uint32_t a, uint32_t b, uint32_t c) {
    sum = a ^ b ^ c;
    carry = (a & b) | (a & c) | (b & c);
}

// Bit-sliced counter: c[b] is the 2^b digit of 32 independent counts (<= 255).
struct SlicedCounter {
    uint32_t c[8];
    __device__ __forceinline__ void clear() {
#pragma unroll
        for (int b = 0; b < 8; ++b) c[b] = 0u;
    }
    // add `x` (a bit-plane of weight 2^from) with ripple carry into planes from..7
    template <int FROM>
    __device__ __forceinline__ void add_plane(uint32_t x) {
#pragma unroll
        for (int b = FROM; b < 8; ++b) {
            const uint32_t t = c[b] & x;
            c[b] ^= x;
            x = t;
        }
    }
    // add 8 one-bit words: 7 CSAs down to one weight-8 plane (+ the running 1/2/4 planes)
    __device__ __forceinline__ void add8(const uint32_t (&x)[8]) {
        uint32_t t2a, t2b, t2c, t2d, t4a, t4b, t8;
        csa(t2a, c[0], c[0], x[0], x[1]);
        csa(t2b, c[0], c[0], x[2], x[3]);
        csa(t4a, c[1], c[1], t2a, t2b);
        csa(t2c, c[0], c[0], x[4], x[5]);
        csa(t2d, c[0], c[0], x[6], x[7]);
        csa(t4b, c[1], c[1], t2c, t2d);
        csa(t8, c[2], c[2], t4a, t4b);
        add_plane<3>(t8);
    }
};

// c += x where x is a bit-sliced number of up to 8 planes (NEXT-1: adding a group's partial count)
__device__ __forceinline__ void sliced_add(SlicedCounter &sc, const uint32_t (&x)[8]) {
    uint32_t carry = 0u;
#pragma unroll
    for (int b = 0; b < 8; ++b) {
        const uint32_t a = sc.c[b];
        sc.c[b] = a ^ x[b] ^ carry;
        carry = (a & x[b]) | (a & carry) | (x[b] & carry);
    }
}

// gt = (a > b) bitwise over 32 lanes; a has 8 planes, b has 9 planes (b may exceed 255)
__device__ __forceinline__ uint32_t sliced_gt(const uint32_t (&a)[8], const uint32_t (&b)[9]) {
    uint32_t gt = 0u, eq = ~b[8];            // a's plane 8 is zero: if b[8] is set, a < b
#pragma unroll
    for (int k = 7; k >= 0; --k) {
        gt |= eq & a[k] & ~b[k];
        eq &= ~(a[k] ^ b[k]);
    }
    return gt;
}

// b = a + m (m <= 255 constant across lanes), 9 planes
__device__ __forceinline__ void sliced_add_const(const uint32_t (&a)[8], int m, uint32_t (&b)[9]) {
    uint32_t carry = 0u;
#pragma unroll
    for (int k = 0; k < 8; ++k) {
        const uint32_t mk = ((m >> k) & 1) ? 0xffffffffu : 0u;
        b[k] = a[k] ^ mk ^ carry;
        carry = (a[k] & mk) | (a[k] & carry) | (mk & carry);
    }
    b[8] = carry;
}

__device__ __forceinline__ void const_planes(int v, uint32_t (&b)[9]) {
#pragma unroll
    for (int k = 0; k < 9; ++k) b[k] = ((v >> k) & 1) ? 0xffffffffu : 0u;
}

// Stream the W words of word position k of both planes into two sliced counters: 16 workers per round,
// i.e. up to 32 independent loads in flight per thread (a thread walks W serially, so the depth of
// each round, not the thread count, is what hides the HBM latency at large fan-in). Small fan-in (W <= 16)
// uses 8 per round: fewer registers, twice the resident CTAs, fewer waves of the latency-bound prologue.
template <bool TERNARY, int ROUND>
__device__ __forceinline__ void count_words2(const uint32_t *__restrict__ P, const uint32_t *__restrict__ N,
                                             int64_t stride, int W, SlicedCounter &cp, SlicedCounter &cn) {
    static_assert(ROUND == 8 || ROUND == 16, "workers per round");
    cp.clear();
    cn.clear();
    for (int w = 0; w < W; w += ROUND) {
        uint32_t xp[ROUND], xn[ROUND];
#pragma unroll
        for (int i = 0; i < ROUND; ++i) {
            const bool in = w + i < W;
            xp[i] = in ? __ldcs(P + (size_t)(w + i) * stride) : 0u;
            xn[i] = (TERNARY && in) ? __ldcs(N + (size_t)(w + i) * stride) : 0u;
        }
#pragma unroll
        for (int h = 0; h < ROUND; h += 8) {
            cp.add8(reinterpret_cast<const uint32_t(&)[8]>(xp[h]));
            if (TERNARY) cn.add8(reinterpret_cast<const uint32_t(&)[8]>(xn[h]));
        }
    }
}

// ---------------------------------------------------------------------------------------------
// The three pieces every a3 kernel shares: where a word position lives, the vote, the write-back.
// ---------------------------------------------------------------------------------------------
struct WordMeta {
    int nvalid;        // elements of the word that exist (0: no such word), 32 except in a tensor's last word
    int li;            // index of the word's tensor in the plan's list of L tensors, -1: no such word
    int64_t obase;     // bucket position of the word's first element
};

__device__ __forceinline__ LtRec load_rec(const LtRec *r) {
    const longlong2 *q = reinterpret_cast<const longlong2 *>(r);
    const longlong2 a = __ldg(q), b = __ldg(q + 1), c = __ldg(q + 2);
    return LtRec{a.x, a.y, b.x, b.y, c.x, c.y};
}
__device__ __forceinline__ WordMeta word_meta(const ReduceParams &p, const PlanView &pv, int nL, int64_t Wd, int64_t k) {
    WordMeta m{0, -1, 0};
    if (k < Wd) {
        const int li = upper_tensor<int64_t>(pv.lt_woff, nL, k);
        const LtRec r = load_rec(pv.lt_rec + li);              // one 48-byte record instead of four dependent lookups
        const int64_t i0 = (k - r.kfirst) * 32;                // tensor-relative first element
        const int64_t rem = r.len - i0;
        m.nvalid = rem >= 32 ? 32 : (int)rem;
        m.obase = r.off + i0;
        m.li = li;
    }
    return m;
}

// The tensor a warp's previous 32 words fell into, kept in registers: consecutive units of a warp mostly
// stay inside one tensor (the low-bit tensors are the big ones), and then neither the lookups above nor the
// per-tensor scale (each a chain of dependent L2 round trips) are repeated.
struct TensorCache {
    int li;                    // -1: empty
    int64_t kfirst, kend;      // word range [kfirst, kend) of the tensor
    int64_t len, off;
    float S;
};

// true (warp-uniform) iff the 32 words k - lane .. k - lane + 31 all belong to the cached tensor
__device__ __forceinline__ bool cached_meta(const TensorCache &c, int64_t k, int lane, WordMeta &m) {
    const int64_t k0 = k - lane;
    if (c.li < 0 || k0 < c.kfirst || k0 + 32 > c.kend) return false;
    const int64_t i0 = (k - c.kfirst) * 32;
    const int64_t rem = c.len - i0;
    m.nvalid = rem >= 32 ? 32 : (int)rem;
    m.obase = c.off + i0;
    m.li = c.li;
    return true;
}

// majority vote with margin on 32 bit-sliced counts: masks of the elements that decode to +S_t and -S_t
__device__ __forceinline__ void vote_masks(const ReduceParams &p, int W, const SlicedCounter &cpv, const SlicedCounter &cnv,
                                           int nvalid, uint32_t &dpos, uint32_t &dneg) {
    if (p.ternary) {
        // d+ = cpos > cneg + m ; d- = cneg > cpos + m      (D = cpos - cneg vs margin)
        uint32_t b[9];
        sliced_add_const(cnv.c, p.margin, b);
        dpos = sliced_gt(cpv.c, b);
        sliced_add_const(cpv.c, p.margin, b);
        dneg = sliced_gt(cnv.c, b);
    } else {
        // G-Binary: cneg = W - cpos; D = 2 cpos - W.  d+ : cpos > floor((W+m)/2);
        // d- : cpos < ceil((W-m)/2)  (never if W <= m)
        uint32_t b[9], a9[9];
        const_planes((W + p.margin) >> 1, b);
        dpos = sliced_gt(cpv.c, b);
        const int k2 = (W > p.margin) ? (W - p.margin + 1) >> 1 : 0;
        // k2 > cpos  <=>  const(k2) > cpos : compare with roles swapped
        uint32_t ka[8];
#pragma unroll
        for (int q = 0; q < 8; ++q) { ka[q] = ((k2 >> q) & 1) ? 0xffffffffu : 0u; a9[q] = cpv.c[q]; }
        a9[8] = 0u;
        dneg = sliced_gt(ka, a9);
    }
    const uint32_t vmask = nvalid >= 32 ? 0xffffffffu : ((1u << nvalid) - 1u);
    dpos &= vmask;
    dneg &= vmask;
}

// A (converged) warp holding 32 consecutive word positions k0 .. k0+31 (lane = word) computes the scales of
// the tensors those words touch (none when the warp is still inside the cached tensor), publishes the scale of a
// tensor whose first word it holds, and returns the scale of this lane's word.
__device__ __forceinline__ float warp_scales(const ReduceParams &p, const PlanView &pv, int W, int lane, int64_t k,
                                             const WordMeta &m, bool hit, TensorCache &tc) {
    float S = tc.S;
    if (!hit) {
        S = 0.f;
        // one cooperative scale per distinct tensor among the warp's words (usually one)
        const int li_lo = __shfl_sync(0xffffffffu, m.li, 0);
        int li_hi = m.li;
#pragma unroll
        for (int d = 16; d >= 1; d >>= 1) li_hi = max(li_hi, __shfl_xor_sync(0xffffffffu, li_hi, d));
        for (int li = li_lo; li >= 0 && li <= li_hi; ++li) {
            const LtRec r = load_rec(pv.lt_rec + li);
            const int t = (int)r.t;
            const float St = warp_tensor_scale(p.abs_sum, W, p.T, t, r.len, lane);
            if (m.li == li) S = St;
            if (lane == 0 && r.kfirst >= k && r.kfirst < k + 32) {  // this warp holds the tensor's first word
                pv.scale[t] = St;
                if (p.scale_out) p.scale_out[t] = St;
            }
            if (li == li_hi) {                                      // remember the last tensor seen (warp-uniform)
                tc.li = li;
                tc.kfirst = r.kfirst;
                tc.kend = r.kend;
                tc.len = r.len;
                tc.off = r.off;
                tc.S = St;
            }
        }
    }
    return S;
}

// The warp writes out = S_t * d for its 32 words (and the counts, when asked for).
template <bool WRITE_COUNTS>
__device__ __forceinline__ void write_back(const ReduceParams &p, int W, int lane, const WordMeta &m, float S,
                                           uint32_t dpos, uint32_t dneg, const SlicedCounter &cpv,
                                           const SlicedCounter &cnv, const float4 *s_dtab) {
    // Fast write-back: the warp's 32 words are 1024 consecutive, 16-byte-aligned elements of ONE tensor.
    // Each thread turns its two masks into 8 direction bytes (low nibble +, high nibble -); a byte
    // indexes a shared-memory table of float4 directions, and every store writes 512 contiguous bytes.
    // (ONE tensor: two low-bit tensors that are adjacent in the bucket, the first a whole number of words long, are
    // contiguous in `out` too, but each has its own scale)
    const int64_t ob0 = __shfl_sync(0xffffffffu, m.obase, 0);
    const int li0 = __shfl_sync(0xffffffffu, m.li, 0);
    const bool fast = !WRITE_COUNTS &&
                      __all_sync(0xffffffffu, m.nvalid == 32 && m.obase == ob0 + 32 * lane && m.li == li0) &&
                      ((ob0 & 3) == 0);
    if (fast) {
        auto spread = [](uint32_t x) {           // 4 nibbles of a 16-bit value -> low nibbles of 4 bytes
            x = (x | (x << 8)) & 0x00ff00ffu;
            return (x | (x << 4)) & 0x0f0f0f0fu;
        };
        const uint32_t lo = spread(dpos & 0xffffu) | (spread(dneg & 0xffffu) << 4);
        const uint32_t hi = spread(dpos >> 16) | (spread(dneg >> 16) << 4);
        const float S0 = __shfl_sync(0xffffffffu, S, 0);
#pragma unroll
        for (int j = 0; j < 8; ++j) {
            // store j covers elements j*128 + lane*4 .. +3 = byte (lane & 7) of thread j*4 + (lane >> 3)
            const int src = j * 4 + (lane >> 3);
            const uint32_t wl = __shfl_sync(0xffffffffu, lo, src), wh = __shfl_sync(0xffffffffu, hi, src);
            const uint32_t d = (((lane & 4) ? wh : wl) >> (8 * (lane & 3))) & 0xffu;
            float4 v = s_dtab[d];
            v.x = __fmul_rn(S0, v.x); v.y = __fmul_rn(S0, v.y);
            v.z = __fmul_rn(S0, v.z); v.w = __fmul_rn(S0, v.w);
            __stcs(reinterpret_cast<float4 *>(p.out + ob0 + j * 128 + lane * 4), v);
        }
        return;
    }
    // general write-back (tensor boundaries, ragged words, count outputs): iteration j handles the word of lane j
#pragma unroll 4
    for (int j = 0; j < 32; ++j) {
        const int nv = __shfl_sync(0xffffffffu, m.nvalid, j);
        if (nv == 0) continue;                               // warp-uniform
        const uint32_t dp = __shfl_sync(0xffffffffu, dpos, j);
        const uint32_t dn = __shfl_sync(0xffffffffu, dneg, j);
        const int64_t ob = __shfl_sync(0xffffffffu, m.obase, j);
        const float Sj = __shfl_sync(0xffffffffu, S, j);
        const int d = (int)((dp >> lane) & 1u) - (int)((dn >> lane) & 1u);
        if (lane < nv) p.out[ob + lane] = __fmul_rn(Sj, (float)d);
        if (WRITE_COUNTS) {
            uint32_t c1 = 0u, c2 = 0u;
#pragma unroll
            for (int b = 0; b < 8; ++b) {
                c1 |= ((__shfl_sync(0xffffffffu, cpv.c[b], j) >> lane) & 1u) << b;
                c2 |= ((__shfl_sync(0xffffffffu, cnv.c[b], j) >> lane) & 1u) << b;
            }
            if (!p.ternary) c2 = (uint32_t)W - c1;
            if (lane < nv) {
                if (p.cpos) p.cpos[ob + lane] = (uint8_t)c1;
                if (p.cneg) p.cneg[ob + lane] = (uint8_t)c2;
            }
        }
    }
}

__device__ __forceinline__ void fill_direction_table(float4 *s_dtab, int i) {   // i in [0, 256)
    s_dtab[i] = make_float4((float)((i & 1) - ((i >> 4) & 1)), (float)(((i >> 1) & 1) - ((i >> 5) & 1)),
                            (float)(((i >> 2) & 1) - ((i >> 6) & 1)), (float)(((i >> 3) & 1) - ((i >> 7) & 1)));
}

// CTA 0 publishes the scales of the tensors that own no word (the others are published by the warp that
// holds the tensor's first word)
__device__ __forceinline__ void publish_wordless_scales(const ReduceParams &p, const PlanView &pv, int W, int nthreads) {
    if (blockIdx.x != 0) return;
    for (int t = threadIdx.x; t < p.T; t += nthreads) {
        const bool isL = p.route[t] == NF_ROUTE_L;
        if (isL && p.len[t] > 0) continue;
        const float S0 = isL ? tensor_scale(p.abs_sum, W, p.T, t, p.len[t]) : 0.f;
        pv.scale[t] = S0;
        if (p.scale_out) p.scale_out[t] = S0;
    }
}

// ---------------------------------------------------------------------------------------------
// a3, register-staged variant: one thread walks the W words of its word position with plain loads.
// Used for planes / partial-count planes the bulk-copy engine cannot take (rows not 16-byte aligned).
// resident CTAs per SM of the deep-round variant: 3 (80 registers, no spills) measured 20-25 % faster than 2
// at W >= 32 (a thread walks W serially, so the bytes in flight per SM come from occupancy)
// ---------------------------------------------------------------------------------------------
#ifndef NF_CR_MINB
#define NF_CR_MINB 3
#endif
template <bool WRITE_COUNTS, bool MERGE, int ROUND>
__global__ void __launch_bounds__(kRThreads, ROUND == 8 ? 4 : NF_CR_MINB) count_reduce_kernel(const ReduceParams p) {
    __shared__ float4 s_dtab[256];          // byte of 4 (+,-) flag pairs -> float4 of directions in {-1, 0, +1}
    fill_direction_table(s_dtab, threadIdx.x);      // kRThreads == 256
    const PlanView pv = plan_view(p.plan, p.T);
    if (pv.hdr->magic != kPlanMagic || pv.hdr->status != NF_OK) return;
    const int64_t Wd = pv.hdr->Wd;
    if (MERGE ? Wd > p.count_stride : Wd > p.plane_stride) return;     // rows shorter than the packed words: nothing is read
    const int nL = pv.hdr->nL;
    const int lane = threadIdx.x & 31;
    const int W = p.W;
    const int64_t n_chunks = (Wd + kRThreads - 1) / kRThreads;
    __syncthreads();                        // direction table
    // Scales are computed warp by warp for the tensors a warp's 32 words touch (no CTA-wide serial
    // prologue: at W = 128 a single thread summing 128 L2 round trips per tensor used to stall every
    // CTA at a barrier).
    publish_wordless_scales(p, pv, W, kRThreads);
    TensorCache tc{-1, 0, 0, 0, 0, 0.f};

    for (int64_t chunk = blockIdx.x; chunk < n_chunks; chunk += gridDim.x) {
        const int64_t k = chunk * kRThreads + threadIdx.x;      // global word position
        uint32_t dpos = 0u, dneg = 0u;
        SlicedCounter cpv, cnv;
        cpv.clear(); cnv.clear();
        WordMeta m{0, -1, 0};
        const bool hit = cached_meta(tc, k, lane, m);
        if (!hit) m = word_meta(p, pv, nL, Wd, k);
        if (k < Wd) {
            if (MERGE) {
                // NEXT-1 level 2: sum of the G groups' bit-sliced partial counts
                // (two groups' planes in flight per round: up to 32 independent loads per thread)
                for (int g = 0; g < p.G; g += 2) {
                    uint32_t xp[2][8], xn[2][8];
#pragma unroll
                    for (int u = 0; u < 2; ++u)
#pragma unroll
                        for (int b = 0; b < 8; ++b) {
                            const bool in = b < p.B && g + u < p.G;
                            const size_t o = ((size_t)(g + u) * p.B + b) * p.count_stride + k;
                            xp[u][b] = in ? __ldcs(p.cnt_pos + o) : 0u;
                            xn[u][b] = (in && p.ternary) ? __ldcs(p.cnt_neg + o) : 0u;
                        }
#pragma unroll
                    for (int u = 0; u < 2; ++u) {
                        sliced_add(cpv, xp[u]);
                        if (p.ternary) sliced_add(cnv, xn[u]);
                    }
                }
            } else if (p.ternary) {
                count_words2<true, ROUND>(p.P + k, p.N + k, p.plane_stride, W, cpv, cnv);
            } else {
                count_words2<false, ROUND>(p.P + k, p.N, p.plane_stride, W, cpv, cnv);
            }
            vote_masks(p, W, cpv, cnv, m.nvalid, dpos, dneg);
        }
        const float S = warp_scales(p, pv, W, lane, k, m, hit, tc);
        write_back<WRITE_COUNTS>(p, W, lane, m, S, dpos, dneg, cpv, cnv, s_dtab);
    }
}

// ---------------------------------------------------------------------------------------------
// a3, ring variant (the default). The endpoint's service rate under fan-in W is an
// HBM-streaming problem: p*W rows of packed words per word position. A thread that walks its W words
// with plain loads has the bytes in flight capped by its registers; here a producer lane issues
// one-dimensional bulk async copies (cp.async.bulk, the TMA engine; 1 KB = 256 words of one worker's
// plane per copy, L2 evict-first: the planes are read once) into a ring of stages of 16 rows that
// complete on the stage's "full" mbarrier, and 8 consumer warps (thread = word position) add each
// stage into their bit-sliced counters (conflict-free LDS.32), release it on the "empty" mbarrier
// and, once the W workers are in, vote and write back exactly as above. A stage holds 8 workers'
// P rows and N rows (G-Ternary) or 16 workers' P rows (G-Binary). The bytes in flight per SM
// (NF_CRQ_MINB CTAs x NF_CRQ_STAGES x 16 KB) do not depend on registers or on W; the write-back of
// unit u overlaps the copies of units u+1 ...
// ---------------------------------------------------------------------------------------------
#ifndef NF_CRQ_STAGES
#define NF_CRQ_STAGES 4
#endif
#ifndef NF_CRQ_MINB
#define NF_CRQ_MINB 3
#endif
#ifndef NF_CRQ_WORDS
#define NF_CRQ_WORDS 256
#endif
constexpr int kQWords = NF_CRQ_WORDS;              // word positions per unit = consumer threads
constexpr int kQRows = 16;                         // rows (worker, plane) per stage
constexpr int kQStageWords = kQRows * kQWords;     // 16 KB
constexpr int kQStages = NF_CRQ_STAGES;
constexpr int kQThreads = kQWords + 32;            // + producer warp
constexpr int kQHdr = 256 + 4096;                  // mbarriers, direction table
constexpr size_t kQSmem = kQHdr + (size_t)kQStages * kQStageWords * 4;
static_assert(2 * kQStages * 8 <= 256, "mbarriers fit the header");

template <bool WRITE_COUNTS, bool MERGE, bool PARTIAL>
__global__ void __launch_bounds__(kQThreads, NF_CRQ_MINB) count_reduce_ring_kernel(const __grid_constant__ ReduceParams p) {
    extern __shared__ __align__(128) unsigned char q_smem[];
    uint64_t *full = reinterpret_cast<uint64_t *>(q_smem);
    uint64_t *empty = full + kQStages;
    float4 *s_dtab = reinterpret_cast<float4 *>(q_smem + 256);
    uint32_t *ring = reinterpret_cast<uint32_t *>(q_smem + kQHdr);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    pdl_launch_dependents();                 // the next kernel's launch and prologue may overlap this kernel
    if (tid == 0) {
        for (int s = 0; s < kQStages; ++s) { mbar_init(full + s, 1); mbar_init(empty + s, kQWords / 32); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    for (int i = tid; i < 256; i += kQThreads) fill_direction_table(s_dtab, i);
    __syncthreads();
    pdl_wait();                              // everything above touched shared memory only
    // PARTIAL (NEXT-1 level 1, "node-local counting"): the bit-sliced counts of this group's W workers are
    // the OUTPUT (B planes per sign); no plan, no tensors, no vote: the word count comes with the call
    const PlanView pv = PARTIAL ? PlanView{} : plan_view(p.plan, p.T);
    if (!PARTIAL && (pv.hdr->magic != kPlanMagic || pv.hdr->status != NF_OK)) return;
    const int64_t Wd = PARTIAL ? p.part_Wd : pv.hdr->Wd;
    if (MERGE ? Wd > p.count_stride : Wd > p.plane_stride) return;     // rows shorter than the packed words: nothing is read
    const int nL = PARTIAL ? 0 : pv.hdr->nL;
    const int W = p.W;
    const bool ternary = p.ternary != 0;
    const int64_t n_units = (Wd + kQWords - 1) / kQWords;
    const int wadv = ternary ? 8 : 16;             // workers per stage
    // stages per unit. MERGE (NEXT-1 level 2, PAPER L243 / L267): one stage per group, rows 0..B-1 = the B bit-planes
    // of the group's partial pos-count, rows 8..8+B-1 = of its neg-count
    const int n_stg = MERGE ? p.G : (W + wadv - 1) / wadv;

    if (warp == kQWords / 32) {
        // ---- producer ----
        if (lane != 0) return;
        const uint64_t pol = policy_evict_first();
        int st = 0;
        uint32_t ph = 0;
        for (int64_t unit = blockIdx.x; unit < n_units; unit += gridDim.x) {
            const int64_t k0 = unit * kQWords;
            const int64_t left = Wd - k0;
            // whole 16-byte chunks (plane_stride is a multiple of 4 words: the last chunk stays inside the row)
            const uint32_t bytes = (uint32_t)(((left >= kQWords ? kQWords : (int)left) + 3) & ~3) * 4u;
            for (int g = 0; g < n_stg; ++g) {
                const int w0 = g * wadv;
                const int nw = min(wadv, W - w0);
                mbar_wait(empty + st, ph ^ 1u);                        // first lap: passes at once
                uint32_t *dst = ring + (size_t)st * kQStageWords;
                if (MERGE) {
                    mbar_expect_tx(full + st, (ternary ? 2u : 1u) * (uint32_t)p.B * bytes);
                    for (int b = 0; b < p.B; ++b) {
                        const size_t o = ((size_t)g * p.B + b) * p.count_stride + k0;
                        bulk_g2s(dst + b * kQWords, p.cnt_pos + o, bytes, full + st, pol);
                        if (ternary) bulk_g2s(dst + (8 + b) * kQWords, p.cnt_neg + o, bytes, full + st, pol);
                    }
                } else if (ternary) {
                    mbar_expect_tx(full + st, 2u * (uint32_t)nw * bytes);
                    for (int w = 0; w < nw; ++w) {
                        const size_t o = (size_t)(w0 + w) * p.plane_stride + k0;
                        bulk_g2s(dst + w * kQWords, p.P + o, bytes, full + st, pol);
                        bulk_g2s(dst + (8 + w) * kQWords, p.N + o, bytes, full + st, pol);
                    }
                } else {
                    mbar_expect_tx(full + st, (uint32_t)nw * bytes);
                    for (int w = 0; w < nw; ++w)
                        bulk_g2s(dst + w * kQWords, p.P + (size_t)(w0 + w) * p.plane_stride + k0, bytes, full + st, pol);
                }
                if (++st == kQStages) { st = 0; ph ^= 1u; }
            }
        }
        return;
    }

    // ---- consumers: thread = word position ----
    if (!PARTIAL) publish_wordless_scales(p, pv, W, kQWords);
    int st = 0;
    uint32_t ph = 0;
    TensorCache tc{-1, 0, 0, 0, 0, 0.f};
    for (int64_t unit = blockIdx.x; unit < n_units; unit += gridDim.x) {
        const int64_t k = unit * kQWords + tid;
        WordMeta m{0, -1, 0};
        float S = 0.f;
        if (!PARTIAL) {
            const bool hit = cached_meta(tc, k, lane, m);
            if (!hit) m = word_meta(p, pv, nL, Wd, k);                 // overlaps the copies in flight,
            S = warp_scales(p, pv, W, lane, k, m, hit, tc);            // and so does the chain of W abs-sums
        }
        SlicedCounter cpv, cnv;
        cpv.clear(); cnv.clear();
        for (int g = 0; g < n_stg; ++g) {
            const int left = W - g * wadv;                             // workers from this stage on
            const int na = MERGE ? p.B : min(8, left);                 // rows 0..7 in use
            const int nb = MERGE ? (ternary ? p.B : 0)
                                 : (ternary ? na : min(8, left - 8));  // rows 8..15 in use (may be <= 0)
            mbar_wait(full + st, ph);
            const uint32_t *src = ring + (size_t)st * kQStageWords + tid;
            uint32_t xa[8], xb[8];
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                xa[i] = i < na ? src[i * kQWords] : 0u;
                xb[i] = i < nb ? src[(8 + i) * kQWords] : 0u;
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(empty + st);                    // every lane's reads of the stage are done
            if (MERGE) {
                sliced_add(cpv, xa);                                   // + the group's bit-sliced partial count
                if (ternary) sliced_add(cnv, xb);
            } else {
                cpv.add8(xa);
                if (ternary) cnv.add8(xb);
                else if (nb > 0) cpv.add8(xb);
            }
            if (++st == kQStages) { st = 0; ph ^= 1u; }
        }
        if (PARTIAL) {
            if (k < Wd) {
#pragma unroll
                for (int b = 0; b < 8; ++b) {
                    if (b >= p.B) break;
                    p.part_pos[(size_t)b * p.count_stride + k] = cpv.c[b];
                    if (ternary) p.part_neg[(size_t)b * p.count_stride + k] = cnv.c[b];
                }
            }
            continue;
        }
        uint32_t dpos = 0u, dneg = 0u;
        if (k < Wd) vote_masks(p, W, cpv, cnv, m.nvalid, dpos, dneg);
        write_back<WRITE_COUNTS>(p, W, lane, m, S, dpos, dneg, cpv, cnv, s_dtab);
    }
}

// NEXT-1 level 1 ("node-local counting", L267): the bit-sliced per-position counts of one
// group of Wg workers' packed planes, B planes per sign = the partial-count payload a node sends.
__global__ void __launch_bounds__(kRThreads, 3)
partial_count_kernel(const uint32_t *__restrict__ P, const uint32_t *__restrict__ N, int64_t plane_stride, int Wg,
                     int64_t Wd, int ternary, int B, uint32_t *__restrict__ cnt_pos, uint32_t *__restrict__ cnt_neg,
                     int64_t count_stride) {
    for (int64_t k = (int64_t)blockIdx.x * kRThreads + threadIdx.x; k < Wd; k += (int64_t)gridDim.x * kRThreads) {
        SlicedCounter cp, cn;
        if (ternary) count_words2<true, 16>(P + k, N + k, plane_stride, Wg, cp, cn);
        else count_words2<false, 16>(P + k, N, plane_stride, Wg, cp, cn);
#pragma unroll
        for (int b = 0; b < 8; ++b) {
            if (b >= B) break;
            cnt_pos[(size_t)b * count_stride + k] = cp.c[b];
            if (ternary) cnt_neg[(size_t)b * count_stride + k] = cn.c[b];
        }
    }
}

static int grid_for(int64_t units, int per_sm) {
    int64_t g = (int64_t)device_sm_count() * per_sm;
    if (g > units) g = units;
    return (int)(g < 1 ? 1 : g);
}

template <bool WRITE_COUNTS, bool MERGE, bool PARTIAL>
static cudaError_t launch_ring(const ReduceParams &p, int64_t units, cudaStream_t s) {
    static bool attr_set = false;                    // per template instance
    if (!attr_set) {
        cudaError_t e = cudaFuncSetAttribute(count_reduce_ring_kernel<WRITE_COUNTS, MERGE, PARTIAL>,
                                             cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kQSmem);
        if (e != cudaSuccess) return e;
        attr_set = true;
    }
    const int grid = grid_for(units, NF_CRQ_MINB);
    // programmatic stream serialization: the kernel waits (griddepcontrol.wait) for its predecessor on the stream
    // before it touches global memory; only its launch latency and shared-memory prologue overlap
    cudaError_t e = launch_kernel(count_reduce_ring_kernel<WRITE_COUNTS, MERGE, PARTIAL>, (unsigned)grid, kQThreads, kQSmem, s, true, p);
    return e != cudaSuccess ? e : cudaGetLastError();
}

cudaError_t launch_count_reduce(const ReduceParams &p, int64_t n, cudaStream_t s) {
    const int64_t max_words = n / 32 + p.T;
    const int64_t chunks = (max_words + kRThreads - 1) / kRThreads;
    const int grid = grid_for(chunks, 8);
    const bool counts = p.cpos || p.cneg;
    const bool small = !p.cnt_pos && p.W <= 16;              // shallow rounds, 4 CTAs per SM
    // the bulk copies need 16-byte-aligned rows: P, N are (nf_sign_count_reduce checks), so plane_stride % 4 == 0
    const int64_t units = (max_words + kQWords - 1) / kQWords;
    if (!p.cnt_pos && (p.plane_stride & 3) == 0)
        return counts ? launch_ring<true, false, false>(p, units, s) : launch_ring<false, false, false>(p, units, s);
    // level-2 merge: rows of partial-count planes, same alignment rule
    if (p.cnt_pos && (p.count_stride & 3) == 0 && ((uintptr_t)p.cnt_pos & 15) == 0 &&
        (!p.ternary || ((uintptr_t)p.cnt_neg & 15) == 0))
        return counts ? launch_ring<true, true, false>(p, units, s) : launch_ring<false, true, false>(p, units, s);
    if (p.cnt_pos) {
        if (counts) count_reduce_kernel<true, true, 16><<<grid, kRThreads, 0, s>>>(p);
        else count_reduce_kernel<false, true, 16><<<grid, kRThreads, 0, s>>>(p);
    } else if (small) {
        if (counts) count_reduce_kernel<true, false, 8><<<grid, kRThreads, 0, s>>>(p);
        else count_reduce_kernel<false, false, 8><<<grid, kRThreads, 0, s>>>(p);
    } else {
        if (counts) count_reduce_kernel<true, false, 16><<<grid, kRThreads, 0, s>>>(p);
        else count_reduce_kernel<false, false, 16><<<grid, kRThreads, 0, s>>>(p);
    }
    return cudaGetLastError();
}

cudaError_t launch_partial_count(const uint32_t *P, const uint32_t *N, int64_t plane_stride, int Wg, int64_t Wd,
                                 int ternary, int B, uint32_t *cnt_pos, uint32_t *cnt_neg, int64_t count_stride,
                                 cudaStream_t s) {
    if (Wd <= 0) return cudaSuccess;
    // rows the bulk-copy engine can take (16-byte aligned): the same ring kernel as the flat reduce, the count planes
    // as its output; anything else: the register-staged kernel
    if ((plane_stride & 3) == 0 && ((uintptr_t)P & 15) == 0 && (!ternary || ((uintptr_t)N & 15) == 0)) {
        ReduceParams p{};
        p.P = P; p.N = N; p.plane_stride = plane_stride; p.W = Wg; p.ternary = ternary; p.B = B;
        p.part_pos = cnt_pos; p.part_neg = cnt_neg; p.count_stride = count_stride; p.part_Wd = Wd;
        return launch_ring<false, false, true>(p, (Wd + kQWords - 1) / kQWords, s);
    }
    const int grid = grid_for((Wd + kRThreads - 1) / kRThreads, 8);
    partial_count_kernel<<<grid, kRThreads, 0, s>>>(P, N, plane_stride, Wg, Wd, ternary, B, cnt_pos, cnt_neg, count_stride);
    return cudaGetLastError();
}

}  // namespace nf
