"""CPU ORACLE of NEXT-4: the Supervisor's CUSUM recovery state machine that produces the
`nf_state` flags step a1 reads. TEST INFRASTRUCTURE ONLY (same rules as nf_oracle.c): plain Python, one
step at a time, in the paper's order; shares no code with the product.

PAPER L158: "slack is the tolerated per-step increase in the smoothed training-health signal before
degradation evidence accumulates, and the threshold is the accumulated excess that triggers fallback to
FP32"; L177-179: "monitors a smoothed training-health signal and accumulates degradation evidence with
CUSUM ... fallback, cooldown, and guarded readmission"; L143 (4)/(6): admission, veto; Table 2 (L164-165):
"one-epoch cooldown", "2x post-recovery guard".

Readings (DESIGN.md §2 #15-#19; the paper gives no formulas, so everything below the CUSUM recursion itself
is "parity unpinned by the paper"):
  #15 smoothing: m_0 = the first finite x (a NaN / Inf signal is a fault, reading #18, and never enters the
      smoothed signal), m_k = beta*m_{k-1} + (1-beta)*x_k
  #16 CUSUM (Page's one-sided test, the paper's ref [21]): y_k = m_k - m_{k-1};
      S_k = max(0, S_{k-1} + y_k - slack); alarm iff S_k > threshold
  #17 phases: WARMUP (admitted=0) for warmup_steps steps -> ADMITTED -> alarm -> COOLDOWN (veto=1) for
      cooldown_steps steps -> GUARD (readmitted) for guard_steps steps, an alarm in GUARD re-enters COOLDOWN
      with twice the cooldown -> ADMITTED. S is held at 0 during WARMUP and COOLDOWN and restarts from 0.
  #18 any NaN/Inf count reported for the step is an immediate alarm (also for a non-finite signal)
  #19 capacity_ok is passed through from the caller (NEXT-3's guard)
Pins (tests/test_supervisor_cpu.py): closed-form alarm step of a linear ramp, no alarm for slopes <= slack,
max(0, .) reset, exact cooldown / guard lengths, doubled cooldown, synthetic traces with 3 injected
degradations -> 3/3 detections, 0 false (the style of Table 2's evidence column).
"""
import math

WARMUP, ADMITTED, COOLDOWN, GUARD = 0, 1, 2, 3


class Supervisor:
    def __init__(self, warmup_steps, ema_beta, slack, threshold, cooldown_steps, guard_steps):
        self.warmup_steps, self.beta, self.slack, self.threshold = int(warmup_steps), float(ema_beta), float(slack), float(threshold)
        self.cooldown_steps, self.guard_steps = int(cooldown_steps), int(guard_steps)
        self.phase = WARMUP if self.warmup_steps > 0 else ADMITTED
        self.step_no = 0
        self.ema = None                 # not seeded yet
        self.cusum = 0.0
        self.remaining = self.warmup_steps
        self.detections = 0

    def step(self, signal, nan_count=0, inf_count=0, capacity_ok=1):
        """Consumes the health signal of the step just finished; returns the (admitted, veto, capacity_ok)
        flags for the NEXT bucket route decisions."""
        finite = math.isfinite(signal)
        fault = (nan_count > 0) or (inf_count > 0) or (not finite)
        if finite:
            if self.ema is None:
                self.ema, y = float(signal), 0.0
            else:
                new = self.beta * self.ema + (1.0 - self.beta) * float(signal)
                y = new - self.ema
                self.ema = new
        else:
            y = 0.0
        self.step_no += 1
        alarm = False
        if self.phase in (ADMITTED, GUARD):
            self.cusum = max(0.0, self.cusum + y - self.slack)
            alarm = fault or (self.cusum > self.threshold)
        if self.phase == WARMUP:
            self.remaining -= 1
            if self.remaining <= 0:
                self.phase, self.cusum = ADMITTED, 0.0
        elif self.phase == ADMITTED:
            if alarm:
                self.detections += 1
                self.phase, self.remaining, self.cusum = COOLDOWN, self.cooldown_steps, 0.0
        elif self.phase == COOLDOWN:
            self.remaining -= 1
            if self.remaining <= 0:
                self.cusum = 0.0
                if self.guard_steps > 0:
                    self.phase, self.remaining = GUARD, self.guard_steps
                else:
                    self.phase = ADMITTED
        elif self.phase == GUARD:
            if alarm:
                self.detections += 1
                self.phase, self.remaining, self.cusum = COOLDOWN, 2 * self.cooldown_steps, 0.0
            else:
                self.remaining -= 1
                if self.remaining <= 0:
                    self.phase = ADMITTED
        admitted = 0 if self.phase == WARMUP else 1
        veto = 1 if self.phase == COOLDOWN else 0
        return admitted, veto, int(capacity_ok)
