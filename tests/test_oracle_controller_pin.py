"""Pin of the oracle's step-size controller and error norm (reading R10).

The oracle's adaptive loop (`trace_ray`, `error_norm` in oracle/gp_oracle.cpp) is re-enacted here in
Python from the text of R10 and the Dormand-Prince coefficients as published (Dormand & Prince 1980,
typed below as exact fractions — not read from the oracle): seven stages through the oracle's
right-hand side `orc_rhs` (pinned on its own by tests/test_oracle_metric_pins.py), the scaled
max-norm, fac = 0.9 err^(-1/5) clamped to [0.2, 5], the cap h <= 0.1 r, h0 = 0.1 r_obs.  The oracle's
trajectory dump must show the same accepted states, the same step proposals and the same
accept / reject counts.  Teeth: an L2 / RMS norm, a 0.8 or 0.95 safety factor, clamps 0.1 / 10, or
a cap on r_n instead of r_{n+1} each give a different step sequence on the same ray.
"""
import math
from fractions import Fraction as Fr

import numpy as np
import pytest

import gp_workloads as W
from oracle import oracle as O

C_ = [Fr(0), Fr(1, 5), Fr(3, 10), Fr(4, 5), Fr(8, 9), Fr(1), Fr(1)]
A_ = [[],
      [Fr(1, 5)],
      [Fr(3, 40), Fr(9, 40)],
      [Fr(44, 45), Fr(-56, 15), Fr(32, 9)],
      [Fr(19372, 6561), Fr(-25360, 2187), Fr(64448, 6561), Fr(-212, 729)],
      [Fr(9017, 3168), Fr(-355, 33), Fr(46732, 5247), Fr(49, 176), Fr(-5103, 18656)],
      [Fr(35, 384), Fr(0), Fr(500, 1113), Fr(125, 192), Fr(-2187, 6784), Fr(11, 84)]]
B5 = A_[6] + [Fr(0)]
B4 = [Fr(5179, 57600), Fr(0), Fr(7571, 16695), Fr(393, 640), Fr(-92097, 339200), Fr(187, 2100), Fr(1, 40)]
E_ = [float(b5 - b4) for b5, b4 in zip(B5, B4)]
A = [[float(x) for x in row] for row in A_]
B = [float(x) for x in B5]


def test_published_pair_is_what_the_oracle_uses():
    c, a, b, e = O.dp54_tableau()
    assert np.allclose(c, [float(x) for x in C_], rtol=0, atol=1e-16)
    for i in range(7):
        assert np.allclose(a[i, :i], A[i], rtol=1e-15, atol=0)
    assert np.allclose(b, B, rtol=1e-15, atol=0)
    assert np.allclose(e, E_, rtol=1e-13, atol=1e-18)


def enact(w, alpha, beta, norm="max", safety=0.9, fmin=0.2, fmax=5.0, cap_on="new", max_accepted=10**9):
    """R10 in Python: returns (list of (lambda, y6, h_next) after each accepted step, n_acc, n_rej)."""
    m, cfg = w["metric"], w["cfg"]
    st = O.initial_state(m, w["camera"], alpha, beta)
    pt, pph = st[4], st[7]
    rh, _ = O.radii(m)
    r_cap, r_esc = rh * (1.0 + cfg["eps_capture"]), cfg["r_escape"]

    def F(y):
        return O.rhs(m, [y[0], y[1], y[2], y[3], pt, y[4], y[5], pph])
    y = np.array([st[0], st[1], st[2], st[3], st[5], st[6]])
    lam, h = 0.0, cfg["h_cap_rel"] * st[1]
    k1 = F(y)
    out, n_acc, n_rej = [], 0, 0
    while n_acc < max_accepted:
        k = [k1]
        for i in range(1, 7):
            k.append(F(y + h * sum(A[i][j] * k[j] for j in range(i))))
        ynew = y + h * sum(B[j] * k[j] for j in range(6))
        errv = h * sum(E_[j] * k[j] for j in range(7))
        sc = cfg["atol"] + cfg["rtol"] * np.maximum(np.abs(y), np.abs(ynew))
        err = float(np.max(np.abs(errv) / sc)) if norm == "max" else float(np.sqrt(np.mean((errv / sc) ** 2)))
        fac = fmax if err == 0.0 else safety * err ** -0.2
        if err > 1.0:
            n_rej += 1
            h *= max(fmin, fac)
            continue
        n_acc += 1
        if ynew[1] > r_esc or ynew[1] < r_cap:
            break
        hnext = min(h * min(fmax, max(fmin, fac)), cfg["h_cap_rel"] * (ynew[1] if cap_on == "new" else y[1]))
        lam += h
        y, k1, h = ynew, k[6], hnext
        out.append((lam, y.copy(), h))
    return out, n_acc, n_rej


# escaping, near-critical, captured side at the configs' tolerance; the first again at 1e-6, where the
# error allows steps beyond the cap h <= 0.1 r and the min() of R10 item 3 takes its other branch
RAYS = [("C2", -4.0, 3.0, 1e-10), ("C2", 7.1, -0.4, 1e-10), ("C2", 2.0, 5.3, 1e-10), ("C2", -4.0, 3.0, 1e-6)]


@pytest.mark.parametrize("name,alpha,beta,tol", RAYS)
def test_oracle_step_sequence_is_r10(name, alpha, beta, tol):
    w = W.workload(name)
    w["cfg"].update(rtol=tol, atol=tol)
    rec, path = O.trace_one(w, alpha, beta, path_capacity=5000)
    mine, n_acc, n_rej = enact(w, alpha, beta)
    assert rec["n_accepted"] == n_acc and rec["n_rejected"] == n_rej, (rec["n_accepted"], n_acc, rec["n_rejected"], n_rej)
    assert n_acc > (200 if tol == 1e-10 else 40) and (n_rej >= 1 or tol != 1e-10)
    # path[0] is the initial state, path[i] the state after the i-th accepted (non-terminal) step,
    # the last entry the landed state; columns: lambda, t, r, theta, phi, p_r, p_theta, h_next
    assert len(path) == len(mine) + 2
    assert path[0, 7] == w["cfg"]["h_cap_rel"] * w["camera"]["r_obs"]            # R10 item 4
    for (lam, y, h), row in zip(mine, path[1:-1]):
        assert abs(row[0] - lam) <= 1e-9 * max(1.0, abs(lam))
        assert np.allclose(row[1:7], y, rtol=1e-9, atol=1e-9)
        assert abs(row[7] - h) <= 1e-6 * h, (row[7], h)       # err^(-1/5) carries the rounding of a cancellation
    capped = sum(1 for (_, y, h) in mine if h == w["cfg"]["h_cap_rel"] * y[1])
    free = len(mine) - capped
    assert free > (50 if tol == 1e-10 else -1)
    if tol == 1e-6:
        assert capped > 10, capped                            # the cap branch of the min() is exercised


LOOSE = dict(rtol=1e-6, atol=1e-6, h_cap_rel=1.0)   # first steps far too long: the clamps and the cap bind


@pytest.mark.parametrize("variant,cfg", [(dict(norm="rms"), {}), (dict(safety=0.8), {}), (dict(safety=0.95), {}),
                                         (dict(fmin=0.1, fmax=10.0), LOOSE), (dict(cap_on="old"), dict(rtol=1e-6, atol=1e-6))])
def test_other_controllers_give_other_sequences(variant, cfg):
    """Teeth of the pin above: each plausible alternative reading of "adaptive step control" moves
    the step proposals by far more than the comparison tolerance (and the R10 reading still
    reproduces the oracle under the same settings)."""
    w = W.workload("C2")
    w["cfg"].update(cfg)
    alpha, beta = RAYS[0][1:3]
    same, _, _ = enact(w, alpha, beta, max_accepted=60)
    _, path = O.trace_one(w, alpha, beta, path_capacity=5000)
    other, n_acc, n_rej = enact(w, alpha, beta, max_accepted=250, **variant)
    n = min(len(other), len(path) - 2)
    h_o = path[1:1 + n, 7]
    h_v = np.array([h for (_, _, h) in other[:n]])
    assert (np.abs(h_v - h_o) > 1e-3 * h_o).sum() >= 3, variant
    h_s = np.array([h for (_, _, h) in same])
    assert np.allclose(h_s[:min(n, 59)], h_o[:min(n, 59, len(h_s))], rtol=1e-6)


def test_error_norm_through_single_step():
    """orc_single_step's err against the same max-norm computed here, on one state at several h
    (including steps that must be rejected)."""
    w = W.workload("C2")
    m = w["metric"]
    st = O.initial_state(m, w["camera"], 3.0, -2.0)
    st[1] = 8.0                                          # a state deep in the field (H != 0 is fine here)
    pt, pph = st[4], st[7]

    def F(y):
        return O.rhs(m, [y[0], y[1], y[2], y[3], pt, y[4], y[5], pph])
    y = np.array([st[0], st[1], st[2], st[3], st[5], st[6]])
    errs = []
    for h in (0.05, 0.2, 0.8, 2.0):
        k = [F(y)]
        for i in range(1, 7):
            k.append(F(y + h * sum(A[i][j] * k[j] for j in range(i))))
        ynew = y + h * sum(B[j] * k[j] for j in range(6))
        errv = h * sum(E_[j] * k[j] for j in range(7))
        sc = 1e-10 + 1e-10 * np.maximum(np.abs(y), np.abs(ynew))
        mine = float(np.max(np.abs(errv) / sc))
        out, err = O.single_step(m, 2, st, h, 1e-10, 1e-10)
        assert np.allclose([out[0], out[1], out[2], out[3], out[5], out[6]], ynew, rtol=1e-13, atol=1e-13)
        assert abs(err - mine) <= 1e-6 * mine, (h, err, mine)
        errs.append(err)
    assert errs[0] < 1.0 < errs[-1]
    # fifth-order error estimate: err ~ h^5
    assert 4.0 < math.log(errs[1] / errs[0]) / math.log(4.0) < 6.0
