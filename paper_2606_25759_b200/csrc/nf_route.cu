// nf_route.cu — step a1: per-tensor route codes, packed-word offsets, route counts
// and the tile map ("plan") the streaming kernels walk. PAPER L108 (paths L/F/P), L132/L229
// (route-correctness contract), L143 steps (4)/(6) (admission, veto, capacity guard), L205
// (unmapped => FP32: the caller passes elig = 0).
//
// One CTA of 1024 threads: the work is O(T) with T <= 8192 and must not cost a host round trip;
// tensors are handled in chunks of 1024 with a warp-shuffle block scan carrying three running
// sums (packed words, tiles, L-tensor count). It writes the plan's route-dependent arrays and header
// fields only: the self-cleaning state of the fused path (cursors, completion counters, exact
// accumulators, clean token) is never touched here.
#include <stdlib.h>
#include "nf_internal.cuh"

namespace nf {

constexpr int kRouteThreads = 1024;

struct Scan3 { long long words, tiles, nl; };

__device__ __forceinline__ Scan3 add3(Scan3 a, Scan3 b) {
    return Scan3{a.words + b.words, a.tiles + b.tiles, a.nl + b.nl};
}
__device__ __forceinline__ Scan3 shfl_up3(Scan3 v, int d) {
    return Scan3{__shfl_up_sync(0xffffffffu, v.words, d), __shfl_up_sync(0xffffffffu, v.tiles, d),
                 __shfl_up_sync(0xffffffffu, v.nl, d)};
}

// exclusive block scan; returns the exclusive prefix of v, *total = block sum (same in all threads)
__device__ Scan3 block_exscan3(Scan3 v, Scan3 *total, Scan3 *smem /*[32]*/) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    Scan3 inc = v;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        Scan3 o = shfl_up3(inc, d);
        if (lane >= d) inc = add3(inc, o);
    }
    if (lane == 31) smem[warp] = inc;
    __syncthreads();
    if (warp == 0) {
        Scan3 w = smem[lane];
        Scan3 winc = w;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            Scan3 o = shfl_up3(winc, d);
            if (lane >= d) winc = add3(winc, o);
        }
        smem[lane] = Scan3{winc.words - w.words, winc.tiles - w.tiles, winc.nl - w.nl};  // exclusive
        if (lane == 31) smem[32] = winc;                                                 // total
    }
    __syncthreads();
    Scan3 base = smem[warp];
    *total = smem[32];
    Scan3 ex = Scan3{inc.words - v.words, inc.tiles - v.tiles, inc.nl - v.nl};
    Scan3 r = add3(base, ex);
    __syncthreads();
    return r;
}

__global__ void __launch_bounds__(kRouteThreads, 1)
route_kernel(const int64_t *__restrict__ off, const int64_t *__restrict__ len,
             const uint8_t *__restrict__ elig, int T, int64_t n, nf_state st,
             uint8_t *__restrict__ route, int64_t *__restrict__ woff, int64_t *__restrict__ summary,
             void *plan, int64_t acc_slots, int zero_acc) {
    pdl_launch_dependents();   // the next kernel may start its prologue
    pdl_wait();                // the previous call's kernels still read the plan / accumulators
    __shared__ Scan3 s_scan[33];
    PlanLayout L = plan_layout(T);
    char *pb = (char *)plan;
    PlanHeader *hdr = (PlanHeader *)pb;
    int32_t *tile_prefix = (int32_t *)(pb + L.tile_prefix);
    int32_t *lt_index = (int32_t *)(pb + L.lt_index);
    int64_t *lt_woff = (int64_t *)(pb + L.lt_woff);
    LtRec *lt_rec = (LtRec *)(pb + L.lt_rec);

    // stand-alone use (nf_route_bucket): the exact accumulators the streaming calls add into start from zero
    // (they clear what they use, but the buffer may be fresh); the fused path keeps them clean itself
    if (zero_acc) {
        unsigned long long *acc = (unsigned long long *)(pb + L.acc);
        for (int64_t i = threadIdx.x; i < acc_slots * kAccWords; i += kRouteThreads) acc[i] = 0ull;
    }

    Scan3 carry{0, 0, 0};
    long long nF = 0, nP = 0, e = 0, tot = 0;   // per-thread partials, reduced at the end
    int bad = 0;
    for (int base = 0; base < T; base += kRouteThreads) {
        const int t = base + threadIdx.x;
        Scan3 v{0, 0, 0};
        int r = NF_ROUTE_P;
        long long l = 0;
        if (t < T) {
            const long long o = off[t];
            l = len[t];
            const long long prev_end = (t == 0) ? 0 : off[t - 1] + len[t - 1];
            if (l < 0 || o < prev_end || o + l > n) bad = 1;
            if (l < 0) l = 0;
            // PAPER L143 (4)/(6), L108, L132, L205, L229
            if (!st.admitted) r = NF_ROUTE_P;
            else if (elig[t] == 0) r = NF_ROUTE_P;
            else if (st.veto || !st.capacity_ok) r = NF_ROUTE_F;
            else r = NF_ROUTE_L;
            v.tiles = (l + kTile - 1) / kTile;
            tot += l;
            if (r == NF_ROUTE_L) { v.words = (l + 31) / 32; v.nl = 1; e += l; }
            else if (r == NF_ROUTE_F) ++nF;
            else ++nP;
        }
        Scan3 total;
        Scan3 ex = block_exscan3(v, &total, s_scan);
        ex = add3(ex, carry);
        if (t < T) {
            route[t] = (uint8_t)r;
            woff[t] = (r == NF_ROUTE_L) ? ex.words : -1;
            tile_prefix[t] = (int32_t)ex.tiles;
            if (r == NF_ROUTE_L) {
                lt_index[ex.nl] = t;
                lt_woff[ex.nl] = ex.words;
                lt_rec[ex.nl] = LtRec{t, off[t], l, ex.words, ex.words + v.words, 0};
            }
        }
        carry = add3(carry, total);
    }
    // block-reduce the small tallies through shared memory atomics
    __shared__ unsigned long long s_tal[4];
    __shared__ int s_bad;
    if (threadIdx.x == 0) { s_tal[0] = s_tal[1] = s_tal[2] = s_tal[3] = 0ull; s_bad = 0; }
    __syncthreads();
    // warp sums first: 64-bit shared-memory atomics are compare-and-swap loops, one per thread serialises
    {
        unsigned long long q[4] = {(unsigned long long)nF, (unsigned long long)nP, (unsigned long long)e,
                                   (unsigned long long)tot};
#pragma unroll
        for (int k = 0; k < 4; ++k) {
#pragma unroll
            for (int d = 16; d >= 1; d >>= 1) q[k] += __shfl_xor_sync(0xffffffffu, q[k], d);
            if ((threadIdx.x & 31) == 0 && q[k]) atomicAdd(&s_tal[k], q[k]);
        }
    }
    if (bad) atomicOr(&s_bad, 1);
    __syncthreads();
    if (threadIdx.x == 0) {
        int status = NF_OK;
        if (s_bad || carry.tiles > 0x7fffffffLL) status = NF_ERR_ARG;
        tile_prefix[T] = (int32_t)carry.tiles;
        lt_woff[carry.nl] = carry.words;
        hdr->magic = kPlanMagic;
        hdr->status = status;
        hdr->T = T;
        hdr->nL = (int32_t)carry.nl;
        hdr->n = n;
        hdr->Wd = carry.words;
        hdr->n_tiles = (status == NF_OK) ? (int32_t)carry.tiles : 0;
        hdr->acc_slots = acc_slots;
        summary[NF_SUM_WD] = carry.words;
        summary[NF_SUM_NL] = carry.nl;
        summary[NF_SUM_NF] = (int64_t)s_tal[0];
        summary[NF_SUM_NP] = (int64_t)s_tal[1];
        summary[NF_SUM_E] = (int64_t)s_tal[2];
        summary[NF_SUM_F] = (int64_t)(s_tal[3] - s_tal[2]);
        summary[NF_SUM_TILES] = carry.tiles;
        summary[NF_SUM_STATUS] = status;
    }
}

cudaError_t launch_route(const int64_t *off, const int64_t *len, const uint8_t *elig, int T, int64_t n,
                         nf_state st, uint8_t *route, int64_t *woff, int64_t *summary, void *plan, size_t plan_bytes,
                         int pdl, int zero_acc, cudaStream_t s) {
    const size_t base = plan_layout(T).acc;
    const int64_t acc_slots = plan_bytes > base ? (int64_t)((plan_bytes - base) / (sizeof(unsigned long long) * kAccWords)) : 0;
    cudaError_t e = launch_kernel(route_kernel, 1, kRouteThreads, 0, s, pdl != 0, off, len, elig, T, n, st, route, woff, summary,
                                  plan, acc_slots, zero_acc);
    if (e != cudaSuccess) return e;
    return cudaGetLastError();
}

}  // namespace nf
