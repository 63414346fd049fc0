// nf_guard.cu — NEXT-3, host side: MGTR accounting over a route log and the
// endpoint-capacity guard whose verdict is nf_state.capacity_ok of step a1. DESIGN.md
// readings #14 (bits per element) and #20 (the guard's time model). Pure host arithmetic.
#include <math.h>
#include "nf.h"

extern "C" {

int nf_mgtr(const int64_t *numel, const uint8_t *route, const uint8_t *mode, int64_t n_events,
            double bits_binary, double bits_ternary, int scale_bytes, double *mgtr) {
    if (!mgtr || n_events < 0 || (n_events > 0 && (!numel || !route || !mode))) return NF_ERR_ARG;
    if (!(bits_binary > 0.0) || !(bits_ternary > 0.0) || scale_bytes < 0) return NF_ERR_RANGE;
    double sent = 0.0, fp32_all = 0.0;
    for (int64_t e = 0; e < n_events; ++e) {
        if (numel[e] < 0) return NF_ERR_RANGE;
        const double as_fp32 = 4.0 * (double)numel[e];
        fp32_all += as_fp32;                                   // denominator: the same event replayed as FP32
        if (route[e] == NF_ROUTE_L) {
            if (mode[e] != NF_MODE_GBINARY && mode[e] != NF_MODE_GTERNARY) return NF_ERR_ARG;
            const double bits = mode[e] == NF_MODE_GBINARY ? bits_binary : bits_ternary;
            sent += (double)numel[e] * bits / 8.0 + (double)scale_bytes;
        } else {
            sent += as_fp32;                                   // F and P events count as FP32 bytes (L112)
        }
    }
    *mgtr = fp32_all > 0.0 ? sent / fp32_all : 1.0;
    return NF_OK;
}

int nf_capacity_guard(int64_t n, int nodes, int local_fan_in, double service_rate, double net_bw, int planes,
                      double *t_hier, double *t_fp32) {
    if (n < 0 || nodes < 1 || local_fan_in < 1 || (int64_t)nodes * local_fan_in > 255) return NF_ERR_RANGE;
    if (!(service_rate > 0.0) || !(net_bw > 0.0) || planes < 1 || planes > 2) return NF_ERR_RANGE;
    const double ring = 2.0 * (double)(nodes - 1) / (double)nodes;          // all-reduce bandwidth term
    int B = 0;
    while ((1 << B) <= nodes * local_fan_in) ++B;                           // planes of a count up to W
    const double compact = (double)planes * (double)n / 8.0;                // bytes of one worker's packed update
    const double th = (double)local_fan_in * compact / service_rate + ring * (compact * (double)B) / net_bw;
    const double tf = ring * 4.0 * (double)n / net_bw;
    if (t_hier) *t_hier = th;
    if (t_fp32) *t_fp32 = tf;
    return th < tf ? 1 : 0;
}

}  // extern "C"
