// nf_supervisor.cu — NEXT-4: the Supervisor's recovery controller, host side. It turns the
// per-step training-health signal (and the NaN/Inf tallies of nf_health_stats) into the nf_state flags
// that step a1 (nf_route_bucket / nf_aggregate_bucket) reads. PAPER L158 (slack, threshold), L177-179
// (smoothed health signal, CUSUM, fallback / cooldown / guarded readmission), L143 (4)/(6), Table 2.
// Readings #15-#19 of DESIGN.md §2. Pure host code: no device memory, no stream.
#include <math.h>
#include "nf.h"

namespace {
enum { kWarmup = 0, kAdmitted = 1, kCooldown = 2, kGuard = 3 };
inline void enter_cooldown(nf_supervisor *s, int steps) {
    s->detections += 1;
    s->phase = kCooldown;
    s->remaining = steps;
    s->cusum = 0.0;
}
}  // namespace

extern "C" {

int nf_supervisor_init(nf_supervisor *s, const nf_supervisor_cfg *cfg) {
    if (!s || !cfg) return NF_ERR_ARG;
    if (cfg->warmup_steps < 0 || cfg->cooldown_steps < 1 || cfg->guard_steps < 0) return NF_ERR_RANGE;
    if (!(cfg->ema_beta >= 0.0 && cfg->ema_beta < 1.0) || !(cfg->slack >= 0.0) || !(cfg->threshold > 0.0)) return NF_ERR_RANGE;
    s->cfg = *cfg;
    s->phase = cfg->warmup_steps > 0 ? kWarmup : kAdmitted;
    s->remaining = cfg->warmup_steps;
    s->step = 0;
    s->detections = 0;
    s->ema = NAN;                      // not seeded yet (reading #15: the first FINITE signal seeds it)
    s->cusum = 0.0;
    return NF_OK;
}

int nf_supervisor_step(nf_supervisor *s, double signal, uint64_t nan_count, uint64_t inf_count, int capacity_ok,
                       nf_state *out) {
    if (!s || !out) return NF_ERR_ARG;
    const bool finite = isfinite(signal);
    const bool fault = nan_count != 0 || inf_count != 0 || !finite;           // reading #18
    double y = 0.0;                                                            // increase of the smoothed signal
    if (finite) {
        if (isnan(s->ema)) {
            s->ema = signal;                                                   // reading #15: m_0 = the first finite x
        } else {
            const double m = s->cfg.ema_beta * s->ema + (1.0 - s->cfg.ema_beta) * signal;
            y = m - s->ema;
            s->ema = m;
        }
    }
    s->step += 1;
    bool alarm = false;
    if (s->phase == kAdmitted || s->phase == kGuard) {
        // Page's one-sided CUSUM (reading #16): evidence beyond the tolerated per-step increase
        const double c = s->cusum + y - s->cfg.slack;
        s->cusum = c > 0.0 ? c : 0.0;
        alarm = fault || s->cusum > s->cfg.threshold;
    }
    switch (s->phase) {                                                        // reading #17
        case kWarmup:
            if (--s->remaining <= 0) { s->phase = kAdmitted; s->cusum = 0.0; }
            break;
        case kAdmitted:
            if (alarm) enter_cooldown(s, s->cfg.cooldown_steps);
            break;
        case kCooldown:
            if (--s->remaining <= 0) {
                s->cusum = 0.0;
                if (s->cfg.guard_steps > 0) { s->phase = kGuard; s->remaining = s->cfg.guard_steps; }
                else s->phase = kAdmitted;
            }
            break;
        default:  // kGuard
            if (alarm) enter_cooldown(s, 2 * s->cfg.cooldown_steps);           // Table 2 "2x post-recovery guard"
            else if (--s->remaining <= 0) s->phase = kAdmitted;
            break;
    }
    out->admitted = s->phase == kWarmup ? 0 : 1;
    out->veto = s->phase == kCooldown ? 1 : 0;
    out->capacity_ok = capacity_ok ? 1 : 0;                                    // reading #19
    return NF_OK;
}

}  // extern "C"
