"""`-m "not gpu"`: NEXT-4, the Supervisor's CUSUM recovery state machine (Table 2).
(1) pins of the oracle (oracle/supervisor_oracle.py) against what the mathematics fixes; (2) the product's
host functions nf_supervisor_init / nf_supervisor_step (libnf.so, no GPU needed) step for step against it."""
import math

import numpy as np
import pytest

from oracle import supervisor_oracle as S


def _run(sup, xs, **kw):
    return [sup.step(x, **kw) for x in xs]


def test_linear_ramp_alarm_step_closed_form():
    """beta = 0 (no smoothing): y_k = d per step, S_k = k*(d - slack) -> first alarm at the smallest k with
    k*(d - slack) > threshold, counted from the first admitted step."""
    d, slack, thr = 0.5, 0.125, 2.0
    sup = S.Supervisor(0, 0.0, slack, thr, cooldown_steps=5, guard_steps=0)
    xs = [d * k for k in range(40)]
    flags = _run(sup, xs)
    k_alarm = math.floor(thr / (d - slack)) + 1          # y_0 = 0 on the first step, so +1 step offset
    first_veto = next(i for i, f in enumerate(flags) if f[1] == 1)
    assert first_veto == k_alarm
    assert all(f == (1, 0, 1) for f in flags[:first_veto])


def test_no_alarm_when_increase_within_slack_and_reset_at_zero():
    sup = S.Supervisor(0, 0.0, 0.25, 1.0, 3, 0)
    flags = _run(sup, [0.25 * k for k in range(200)])                 # slope == slack: S stays 0
    assert all(f == (1, 0, 1) for f in flags) and sup.cusum == 0.0 and sup.detections == 0
    # a burst below the threshold followed by a decrease: max(0, .) forgets it
    sup = S.Supervisor(0, 0.0, 0.0, 1.0, 3, 0)
    _run(sup, [0.0, 0.4, 0.8])
    assert sup.cusum == pytest.approx(0.8)
    _run(sup, [-5.0])
    assert sup.cusum == 0.0
    flags = _run(sup, [-4.6, -4.2])                                   # would exceed 1.0 only without the reset
    assert all(f[1] == 0 for f in flags)


def test_phases_warmup_cooldown_guard_lengths():
    sup = S.Supervisor(warmup_steps=4, ema_beta=0.0, slack=0.0, threshold=0.5, cooldown_steps=3, guard_steps=2)
    flags = _run(sup, [1.0] * 4)
    assert [f[0] for f in flags] == [0, 0, 0, 1]                      # admitted after exactly 4 warm-up steps
    flags = _run(sup, [1.0, 2.0])                                     # jump of 1.0 > threshold -> alarm
    assert flags[-1] == (1, 1, 1) and sup.phase == S.COOLDOWN
    flags = _run(sup, [2.0] * 3)
    assert [f[1] for f in flags] == [1, 1, 0] and sup.phase == S.GUARD    # veto for exactly 3 steps in total
    flags = _run(sup, [2.0] * 2)
    assert sup.phase == S.ADMITTED and all(f == (1, 0, 1) for f in flags)
    # alarm during GUARD: cooldown doubles
    sup = S.Supervisor(0, 0.0, 0.0, 0.5, cooldown_steps=2, guard_steps=5)
    _run(sup, [0.0, 1.0])                                             # alarm -> cooldown 2
    _run(sup, [1.0, 1.0])                                             # -> GUARD
    assert sup.phase == S.GUARD
    _run(sup, [2.0])                                                  # alarm in GUARD
    assert sup.phase == S.COOLDOWN and sup.remaining == 4 and sup.detections == 2


def test_fault_counts_trigger_immediately_and_capacity_passthrough():
    sup = S.Supervisor(0, 0.9, 10.0, 100.0, 2, 0)
    assert sup.step(1.0) == (1, 0, 1)
    assert sup.step(1.0, nan_count=3) == (1, 1, 1)
    sup = S.Supervisor(0, 0.9, 10.0, 100.0, 2, 0)
    sup.step(1.0)
    assert sup.step(float("nan")) == (1, 1, 1)
    assert sup.step(1.0, capacity_ok=0)[2] == 0


def test_ema_matches_closed_form():
    beta = 0.8
    sup = S.Supervisor(0, beta, 1e9, 1e9, 1, 0)
    xs = np.random.default_rng(0).standard_normal(50)
    _run(sup, xs)
    m = xs[0]
    for x in xs[1:]:
        m = beta * m + (1 - beta) * x
    assert sup.ema == pytest.approx(m, rel=1e-12)


def _trace(seed, n=600, events=(150, 300, 450)):
    """Noisy decreasing loss with three injected degradations (Table 2's '3/3 true detections, 0 false')."""
    rng = np.random.default_rng(seed)
    x = 2.0 * np.exp(-np.arange(n) / 300.0) + 0.01 * rng.standard_normal(n)
    for e in events:
        x[e:] += 0.5
    return x


@pytest.mark.parametrize("seed", [0, 1, 2])
def test_three_injected_degradations_three_detections_no_false(seed):
    x = _trace(seed)
    sup = S.Supervisor(warmup_steps=20, ema_beta=0.9, slack=0.005, threshold=0.15, cooldown_steps=30, guard_steps=30)
    flags = _run(sup, x)
    veto = np.array([f[1] for f in flags])
    starts = np.flatnonzero(np.diff(np.concatenate([[0], veto])) == 1)
    assert sup.detections == 3 and len(starts) == 3
    for s, e in zip(starts, (150, 300, 450)):
        assert 0 <= s - e <= 15                                       # detected within 15 steps of the onset


# ---- the product's host functions against the oracle -------------------------------------------------
@pytest.fixture(scope="module")
def nf():
    from paper_2606_25759_b200 import build, binding
    build.build()
    return binding


@pytest.mark.parametrize("seed", [0, 3])
def test_library_supervisor_matches_oracle_step_for_step(nf, seed):
    cfg = dict(warmup_steps=20, ema_beta=0.9, slack=0.005, threshold=0.15, cooldown_steps=30, guard_steps=30)
    x = _trace(seed)
    rng = np.random.default_rng(seed)
    nan = (rng.random(len(x)) < 0.005).astype(int)                    # sporadic fault evidence
    cap = (rng.random(len(x)) < 0.95).astype(int)
    ora = S.Supervisor(**cfg)
    lib = nf.Supervisor(**cfg)
    for i in range(len(x)):
        a = ora.step(float(x[i]), nan_count=int(nan[i]), capacity_ok=int(cap[i]))
        b = lib.step(float(x[i]), nan_count=int(nan[i]), capacity_ok=int(cap[i]))
        assert a == b, i
        assert lib.phase == ora.phase and lib.detections == ora.detections
        assert lib.cusum == ora.cusum and lib.ema == ora.ema          # same FP64 operations in the same order


def test_non_finite_first_signals_do_not_seed_the_smoothed_signal(nf):
    """Reading #15: the smoothed signal starts at the FIRST FINITE value. A NaN / Inf at step 0 must not
    leave m at 0 (the next finite x would then look like a jump of (1 - beta) x and, once admitted, like a long climb:
    spurious alarms). Closed form: NaN, Inf, then a constant c for ever -> m = c exactly, y = 0, S = 0, no alarm after
    the faults' own; oracle and library agree step for step."""
    cfg = dict(warmup_steps=0, ema_beta=0.9, slack=0.0, threshold=0.05, cooldown_steps=2, guard_steps=0)
    ora, lib = S.Supervisor(**cfg), nf.Supervisor(**cfg)
    c = 2.5
    xs = [float("nan"), float("inf")] + [c] * 40
    for i, x in enumerate(xs):
        a, b = ora.step(x), lib.step(x)
        assert a == b, i
        if i >= 2:
            assert ora.ema == c and lib.ema == c and ora.cusum == 0.0 and lib.cusum == 0.0
    # the two non-finite signals were faults (reading #18): admitted from the start, so exactly one detection (the
    # second fault falls into the cooldown of the first), none from the constant stretch
    assert ora.detections == 1 and lib.detections == 1
    assert ora.phase == S.ADMITTED and lib.phase == S.ADMITTED
