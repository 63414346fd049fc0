/*
 * nf_oracle.c — CPU ORACLE for the NEURON-Fabric low-bit bucket-aggregation hot path.
 *
 * >>> TEST INFRASTRUCTURE ONLY. <<<
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / `--impl reference`
 * legs may build, load or call this file. The product (paper_2606_25759_b200/ and its CUDA
 * library) never includes, links or imports anything under oracle/, and this file shares no
 * code, header, table or helper with the CUDA path.
 *
 * What it is: a plain, slow, single-threaded, scalar-loop C restatement of what the path
 * computes, step by step in the paper's order. The method is an encoding (sign indicators)
 * + an exact integer aggregation (per-coordinate sign counts) + a scaling, so the oracle is
 * the algorithm itself written out. Citations are PAPER.md line numbers (/root/reference).
 * Where the paper is silent the reading of SURVEY.md §8(c) / DESIGN.md §"Readings" is taken
 * and named "reading #k".
 *
 * Pins (tests/test_oracle_*.py, `-m "not gpu"`):
 *   O1 route  : 16-row truth table from L108/L132/L205/L229; nL+nF+nP=T; 3-state preflight (L207)
 *   O2 pack   : hand-worked bucket (tests/golden/handworked_w4.txt); brute force from floats;
 *               all-positive / all-zero closed forms; P&N==0; padding bits 0; popcount identity
 *   O2 scale  : constant-tensor closed form; numpy abs-sum (library routine)
 *   O3 counts : cpos+cneg+czero=W; brute force; exhaustive 3^W vote table W<=4; permutation invariance
 *   O3 decode : W identical workers => mean|g|*sign(g) (textbook scaled signSGD); W=1; sign flip
 *   O4a fp32  : numpy float32 ordered add; integer-valued exactness; W=1 identity
 *   O4b health: constant closed form; injected NaN/Inf counts; numpy.linalg.norm on finite part
 *   NEXT-1    : hand-worked 2 x 2 split of the same bucket; hierarchical == flat O3 (all splits);
 *               one worker per group => partial planes == packed planes; plane count closed form
 * Readings #3-#9 and #11 (what G-Ternary gating is, tie rule, scale granularity, scale
 * combination, NaN handling) are NOT fixed by the paper: "parity unpinned by the paper" for
 * those choices — they are pinned only by DESIGN.md and sit behind named parameters.
 *
 * Build: gcc -O2 -std=c11 -ffp-contract=off -fno-fast-math -shared -fPIC (oracle/build.py).
 */
#include <math.h>
#include <stdint.h>
#include <string.h>

#define NFO_OK 0
#define NFO_ERR_ARG (-1)
#define NFO_ERR_RANGE (-3)

enum { NFO_ROUTE_P = 0, NFO_ROUTE_L = 1, NFO_ROUTE_F = 2 }; /* L108: paths L / F / P */
enum { NFO_MODE_GBINARY = 1, NFO_MODE_GTERNARY = 2 };       /* L60 */

/* Tensors must lie inside [0,n), in ascending order, without overlap (gaps allowed). */
static int nfo_check_layout(const int64_t *off, const int64_t *len, int T, int64_t n) {
    int64_t end = 0;
    if (T < 0 || n < 0) return NFO_ERR_ARG;
    for (int t = 0; t < T; ++t) {
        if (len[t] < 0 || off[t] < end || off[t] + len[t] > n) return NFO_ERR_ARG;
        end = off[t] + len[t];
    }
    return NFO_OK;
}

/*
 * O1 Route. PAPER L108 (path codes L/F/P), L132 + L229 (route-correctness contract: an
 * FP32-sensitive tensor never takes low-bit; an eligible tensor under an active veto takes
 * FP32 fallback), L143 step (4)/(6) (Commander admission, Supervisor state and the
 * endpoint-capacity guard gate the eligible portion), L205 (unmapped => FP32-only; the caller
 * encodes "unmapped" as elig=0).
 *   not admitted (FP32 warm-up)                 -> P for every tensor
 *   admitted, elig=0                            -> P
 *   admitted, elig=1, veto or !capacity_ok      -> F
 *   admitted, elig=1, no veto, capacity_ok      -> L
 * woff[t] = running sum of ceil(len/32) over L tensors in bucket order (reading #10), -1 if not L.
 * summary = { Wd, nL, nF, nP, e (low-bit elements), f = sum(len) - e }.
 */
int nfo_route_bucket(const int64_t *off, const int64_t *len, const uint8_t *elig, int T, int64_t n,
                     int admitted, int veto, int capacity_ok,
                     uint8_t *route, int64_t *woff, int64_t *summary) {
    int rc = nfo_check_layout(off, len, T, n);
    if (rc != NFO_OK) return rc;
    int64_t words = 0, nL = 0, nF = 0, nP = 0, e = 0, tot = 0;
    for (int t = 0; t < T; ++t) {
        uint8_t r;
        if (!admitted) r = NFO_ROUTE_P;
        else if (elig[t] == 0) r = NFO_ROUTE_P;
        else if (veto || !capacity_ok) r = NFO_ROUTE_F;
        else r = NFO_ROUTE_L;
        route[t] = r;
        tot += len[t];
        if (r == NFO_ROUTE_L) {
            woff[t] = words;
            words += (len[t] + 31) / 32;
            e += len[t];
            ++nL;
        } else {
            woff[t] = -1;
            if (r == NFO_ROUTE_F) ++nF; else ++nP;
        }
    }
    summary[0] = words; summary[1] = nL; summary[2] = nF; summary[3] = nP;
    summary[4] = e; summary[5] = tot - e;
    return NFO_OK;
}

/*
 * O2 Pack. PAPER L211: "records a mean-absolute scale and converts FP32 gradients into dense
 * positive-sign indicators that stand in for packed signs or a ternary payload"; L60: G-Ternary
 * "adds a zero-gating rule that can suppress selected entries before aggregation"; L247
 * "bit-packed updates ... packed machine words".
 * For worker w, L tensor t, element i: x = g_w[off_t+i], tau = tau[t] (0 if tau==NULL):
 *   pos = (x > tau), neg = (x < -tau)   (reading #1/#3: both false for NaN and for +-0 at tau=0)
 *   word k = woff_t + i/32, bit j = i%32 (LSB first, reading #10); P_w[k] |= pos<<j;
 *   G-Ternary only: N_w[k] |= neg<<j. Unused high bits of a tensor's last word stay 0.
 *   A[w][t] = sum_i (double)|x| in index order (numerator of the mean-absolute scale, reading #7).
 * abs_sum is [W][T]; entries of non-L tensors are set to 0.
 */
int nfo_sign_pack(const float *g, int64_t worker_stride, int W, int64_t n,
                  const int64_t *off, const int64_t *len, const uint8_t *route, const int64_t *woff,
                  int T, int mode, const float *tau,
                  uint32_t *P, uint32_t *N, int64_t plane_stride, double *abs_sum) {
    if (W < 1 || W > 255) return NFO_ERR_RANGE;
    if (mode != NFO_MODE_GBINARY && mode != NFO_MODE_GTERNARY) return NFO_ERR_ARG;
    if (nfo_check_layout(off, len, T, n) != NFO_OK || worker_stride < n) return NFO_ERR_ARG;
    for (int w = 0; w < W; ++w) {
        const float *gw = g + (int64_t)w * worker_stride;
        uint32_t *Pw = P + (int64_t)w * plane_stride;
        uint32_t *Nw = (mode == NFO_MODE_GTERNARY) ? N + (int64_t)w * plane_stride : 0;
        for (int t = 0; t < T; ++t) {
            abs_sum[(int64_t)w * T + t] = 0.0;
            if (route[t] != NFO_ROUTE_L) continue;
            int64_t nwords = (len[t] + 31) / 32;
            for (int64_t k = 0; k < nwords; ++k) {
                Pw[woff[t] + k] = 0u;
                if (Nw) Nw[woff[t] + k] = 0u;
            }
            float th = tau ? tau[t] : 0.0f;
            double A = 0.0;
            for (int64_t i = 0; i < len[t]; ++i) {
                float x = gw[off[t] + i];
                int pos = (x > th);
                int neg = (x < -th);
                int64_t k = woff[t] + i / 32;
                int j = (int)(i % 32);
                if (pos) Pw[k] |= (uint32_t)1u << j;
                if (Nw && neg) Nw[k] |= (uint32_t)1u << j;
                A += (double)fabsf(x);
            }
            abs_sum[(int64_t)w * T + t] = A;
        }
    }
    return NFO_OK;
}

/*
 * Reference sign-count straight from the floats, no packed words — the paper's
 * "reference sign-count" mode (L285) and the brute-force side of the count pin.
 * cpos/cneg are [n] uint8 at bucket positions; only positions of L tensors are written.
 */
int nfo_sign_count_reference(const float *g, int64_t worker_stride, int W, int64_t n,
                             const int64_t *off, const int64_t *len, const uint8_t *route, int T,
                             int mode, const float *tau, uint8_t *cpos, uint8_t *cneg) {
    if (W < 1 || W > 255) return NFO_ERR_RANGE;
    if (nfo_check_layout(off, len, T, n) != NFO_OK) return NFO_ERR_ARG;
    for (int t = 0; t < T; ++t) {
        if (route[t] != NFO_ROUTE_L) continue;
        float th = tau ? tau[t] : 0.0f;
        for (int64_t i = 0; i < len[t]; ++i) {
            int cp = 0, cn = 0;
            for (int w = 0; w < W; ++w) {
                float x = g[(int64_t)w * worker_stride + off[t] + i];
                cp += (x > th);
                cn += (x < -th);
            }
            if (mode == NFO_MODE_GBINARY) cn = W - cp; /* reading #2 */
            cpos[off[t] + i] = (uint8_t)cp;
            cneg[off[t] + i] = (uint8_t)cn;
        }
    }
    return NFO_OK;
}

/*
 * O3 Count + decode. PAPER L211: "Ordinary PyTorch collectives then sum these indicators across
 * workers; the hook applies majority voting, optionally applies the G-Ternary zero-gating
 * pattern, and writes the scaled aggregate direction back into the gradient buffer"; L247
 * "sign-count aggregation over bit-packed updates requires recovering per-coordinate sign
 * counts rather than numerically adding packed machine words".
 * For L tensor t, element i (word k = woff_t + i/32, bit j = i%32):
 *   cpos = sum_w bit_j(P_w[k]);  G-Ternary: cneg = sum_w bit_j(N_w[k]);  G-Binary: cneg = W - cpos
 *   czero = W - cpos - cneg;  D = cpos - cneg;  d = (D > m) - (D < -m)     (readings #5, #6, #3)
 *   s_wt = (float)(A[w][t] / len_t);  S_t = (float)( (sum_{w=0..W-1} (double)s_wt) / W )  (#7, #8)
 *   out[off_t+i] = S_t * (float)d                                          (#9, #11: IEEE)
 * Optional outputs: cpos/cneg [n] uint8 (L positions only), scale_out [T] (0 for non-L tensors).
 */
int nfo_sign_count_reduce(const uint32_t *P, const uint32_t *N, int64_t plane_stride, int W,
                          int64_t n, const int64_t *off, const int64_t *len, const uint8_t *route,
                          const int64_t *woff, int T, int mode, int margin, const double *abs_sum,
                          float *out, uint8_t *cpos, uint8_t *cneg, float *scale_out) {
    if (W < 1 || W > 255 || margin < 0 || margin > 255) return NFO_ERR_RANGE;
    if (mode != NFO_MODE_GBINARY && mode != NFO_MODE_GTERNARY) return NFO_ERR_ARG;
    if (nfo_check_layout(off, len, T, n) != NFO_OK) return NFO_ERR_ARG;
    for (int t = 0; t < T; ++t) {
        if (scale_out) scale_out[t] = 0.0f;
        if (route[t] != NFO_ROUTE_L) continue;
        double ssum = 0.0;
        for (int w = 0; w < W; ++w) {
            float s_wt = (float)(abs_sum[(int64_t)w * T + t] / (double)len[t]);
            ssum += (double)s_wt;
        }
        float S = (float)(ssum / (double)W);
        if (scale_out) scale_out[t] = S;
        for (int64_t i = 0; i < len[t]; ++i) {
            int64_t k = woff[t] + i / 32;
            int j = (int)(i % 32);
            int cp = 0, cn = 0;
            for (int w = 0; w < W; ++w) {
                cp += (int)((P[(int64_t)w * plane_stride + k] >> j) & 1u);
                if (mode == NFO_MODE_GTERNARY) cn += (int)((N[(int64_t)w * plane_stride + k] >> j) & 1u);
            }
            if (mode == NFO_MODE_GBINARY) cn = W - cp;
            int D = cp - cn;
            int d = (D > margin) - (D < -margin);
            out[off[t] + i] = S * (float)d;
            if (cpos) cpos[off[t] + i] = (uint8_t)cp;
            if (cneg) cneg[off[t] + i] = (uint8_t)cn;
        }
    }
    return NFO_OK;
}

/*
 * O4a FP32 route. PAPER L50 (all-reduce "by summation or averaging"), L66 (FP32 is the
 * warm-up, recovery and semantic reference path), L144 ("rejected or sensitive slices remain
 * on the FP32 path"). For every P/F tensor, element i:
 *   acc = g_0[i]; for w = 1..W-1: acc = acc + g_w[i]   (float, fixed worker order); out = alpha*acc
 * alpha = 1 -> sum, alpha = 1/W -> DDP mean (reading #9). NaN/Inf propagate. L positions untouched.
 */
int nfo_fp32_reduce(const float *g, int64_t worker_stride, int W, int64_t n,
                    const int64_t *off, const int64_t *len, const uint8_t *route, int T,
                    float alpha, float *out) {
    if (W < 1 || W > 255) return NFO_ERR_RANGE;
    if (nfo_check_layout(off, len, T, n) != NFO_OK || worker_stride < n) return NFO_ERR_ARG;
    for (int t = 0; t < T; ++t) {
        if (route[t] == NFO_ROUTE_L) continue;
        for (int64_t i = 0; i < len[t]; ++i) {
            float acc = g[off[t] + i];
            for (int w = 1; w < W; ++w) {
                float x = g[(int64_t)w * worker_stride + off[t] + i];
                acc = acc + x;
            }
            out[off[t] + i] = alpha * acc;
        }
    }
    return NFO_OK;
}

/*
 * O4b Health statistics. Not defined by the paper (its health signal is the smoothed loss,
 * L158/L177); defined by BASELINE.json north_star step (4): "per-tensor L2 norms, NaN/Inf
 * counts" (reading #13). For replica r, tensor t:
 *   Q = sum over finite x of (double)x*(double)x;  nan = #isnan;  inf = #isinf;  L2 = sqrt(Q).
 * Outputs are [R][T].
 */
int nfo_health_stats(const float *x, int64_t replica_stride, int R, int64_t n,
                     const int64_t *off, const int64_t *len, int T,
                     double *sumsq, uint64_t *nan_cnt, uint64_t *inf_cnt) {
    if (R < 1) return NFO_ERR_RANGE;
    if (nfo_check_layout(off, len, T, n) != NFO_OK || replica_stride < n) return NFO_ERR_ARG;
    for (int r = 0; r < R; ++r) {
        for (int t = 0; t < T; ++t) {
            double Q = 0.0;
            uint64_t cn = 0, ci = 0;
            for (int64_t i = 0; i < len[t]; ++i) {
                float v = x[(int64_t)r * replica_stride + off[t] + i];
                if (isnan(v)) ++cn;
                else if (isinf(v)) ++ci;
                else Q += (double)v * (double)v;
            }
            sumsq[(int64_t)r * T + t] = Q;
            nan_cnt[(int64_t)r * T + t] = cn;
            inf_cnt[(int64_t)r * T + t] = ci;
        }
    }
    return NFO_OK;
}

/*
 * NEXT-1 — two-level hierarchical sign count. PAPER L243: the reducer "aggregates
 * compact worker updates through node-local counting and inter-node partial-count exchange before
 * returning a synchronized aggregate direction"; L267: "performs node-local sign counting,
 * exchanges partial counts, and returns the aggregate direction".
 *
 * Level 1, node-local counting of one group ("node") of Wg workers: for every packed word k and
 * bit j, c = sum_{w < Wg} bit_j(plane_w[k]); the partial count is stored bit-sliced, plane b of
 * word k holding bit b of c at bit position j (the partial-count payload a node sends): B planes,
 * B >= number of bits of Wg (reading: smallest B with 2^B > Wg, nfo_count_planes).
 */
int nfo_count_planes(int Wg) {
    int B = 0;
    while ((1 << B) <= Wg) ++B;
    return B;
}

int nfo_partial_count(const uint32_t *planes, int64_t plane_stride, int Wg, int64_t Wd, int B,
                      uint32_t *cnt, int64_t count_stride) {
    if (Wg < 1 || Wg > 255 || B < 1 || B > 8 || (1 << B) <= Wg) return NFO_ERR_RANGE;
    for (int b = 0; b < B; ++b)
        for (int64_t k = 0; k < Wd; ++k) cnt[(int64_t)b * count_stride + k] = 0u;
    for (int64_t k = 0; k < Wd; ++k)
        for (int j = 0; j < 32; ++j) {
            int c = 0;
            for (int w = 0; w < Wg; ++w) c += (int)((planes[(int64_t)w * plane_stride + k] >> j) & 1u);
            for (int b = 0; b < B; ++b)
                cnt[(int64_t)b * count_stride + k] |= (uint32_t)((c >> b) & 1) << j;
        }
    return NFO_OK;
}

/*
 * Level 2, partial-count merge + decode: cpos = sum over the G groups of their partial counts
 * (read back from the bit-sliced planes), likewise cneg (G-Binary: cneg = W - cpos), then the vote,
 * the scale and the output exactly as in nfo_sign_count_reduce (O3), W = total number of workers,
 * abs_sum[W][T] in global worker order. Layout: cnt[(g*B + b)*count_stride + k].
 */
int nfo_partial_count_merge(const uint32_t *cnt_pos, const uint32_t *cnt_neg, int64_t count_stride, int G,
                            int B, int W, int64_t n, const int64_t *off, const int64_t *len,
                            const uint8_t *route, const int64_t *woff, int T, int mode, int margin,
                            const double *abs_sum, float *out, uint8_t *cpos, uint8_t *cneg,
                            float *scale_out) {
    if (W < 1 || W > 255 || G < 1 || G > W || B < 1 || B > 8 || margin < 0 || margin > 255) return NFO_ERR_RANGE;
    if (mode != NFO_MODE_GBINARY && mode != NFO_MODE_GTERNARY) return NFO_ERR_ARG;
    if (nfo_check_layout(off, len, T, n) != NFO_OK) return NFO_ERR_ARG;
    for (int t = 0; t < T; ++t) {
        if (scale_out) scale_out[t] = 0.0f;
        if (route[t] != NFO_ROUTE_L) continue;
        double ssum = 0.0;
        for (int w = 0; w < W; ++w) {
            float s_wt = (float)(abs_sum[(int64_t)w * T + t] / (double)len[t]);
            ssum += (double)s_wt;
        }
        float S = (float)(ssum / (double)W);
        if (scale_out) scale_out[t] = S;
        for (int64_t i = 0; i < len[t]; ++i) {
            int64_t k = woff[t] + i / 32;
            int j = (int)(i % 32);
            int cp = 0, cn = 0;
            for (int g = 0; g < G; ++g)
                for (int b = 0; b < B; ++b) {
                    cp += (int)((cnt_pos[((int64_t)g * B + b) * count_stride + k] >> j) & 1u) << b;
                    if (mode == NFO_MODE_GTERNARY)
                        cn += (int)((cnt_neg[((int64_t)g * B + b) * count_stride + k] >> j) & 1u) << b;
                }
            if (cp > W || cn > W) return NFO_ERR_RANGE;
            if (mode == NFO_MODE_GBINARY) cn = W - cp;
            int D = cp - cn;
            int d = (D > margin) - (D < -margin);
            out[off[t] + i] = S * (float)d;
            if (cpos) cpos[off[t] + i] = (uint8_t)cp;
            if (cneg) cneg[off[t] + i] = (uint8_t)cn;
        }
    }
    return NFO_OK;
}
