"""Pins of the oracle's orbit integrator (explicit initial states, time-like or null; PAPER.md L286-302,
section 3.2.1 and Fig 1; L719, Fig 11).  CPU only."""
import math

import numpy as np
import pytest
from scipy.integrate import quad, solve_ivp

import gp_workloads as W
from oracle import oracle as O

SCHW = dict(id=W.SCHWARZSCHILD, M=1.0, a=0.0, q=0.0)
KERR = dict(id=W.KERR, M=1.0, a=0.9, q=0.0)
CFG = dict(rtol=1e-11, atol=1e-11, h0=0.1, h_max=5.0, lambda_end=2000.0, n_samples=50)


def schw_circular(r):
    d = math.sqrt(1 - 3 / r)
    return (1 - 2 / r) / d, math.sqrt(r) / d          # E, L per unit mass (M = 1)


def test_schwarzschild_circular_timelike_orbit_closed_form():
    r0 = 10.0
    E, L = schw_circular(r0)
    st = [0.0, r0, math.pi / 2, 0.0, -E, 0.0, 0.0, L]   # physical, future-directed: p_t = -E
    s, status, steps = O.integrate_orbits(SCHW, [st], CFG)
    assert status[0] == 0 and steps[0] < 2000
    lam = s[0, :, 7]
    assert np.array_equal(lam, (np.arange(50) + 1) * 2000.0 / 50)       # samples sit exactly on lambda_k
    assert np.abs(s[0, :, 1] - r0).max() <= 1e-8                          # stays on the circle
    assert np.abs(s[0, :, 2] - math.pi / 2).max() <= 1e-14        # cos(pi/2) is 6e-17, not 0
    assert np.allclose(s[0, :, 3], L / r0 ** 2 * lam, rtol=1e-9)          # dphi/dtau = L / r^2
    assert np.allclose(s[0, :, 0], E / (1 - 2 / r0) * lam, rtol=1e-9)     # dt/dtau = E / (1 - 2M/r)
    assert np.allclose(s[0, :, 6], -1.0, atol=1e-9)                       # 2H = -1: time-like
    # coordinate angular velocity: Kepler's third law holds exactly in Schwarzschild coordinates
    assert s[0, -1, 3] / s[0, -1, 0] == pytest.approx(r0 ** -1.5, rel=1e-9)


def test_kerr_equatorial_circular_orbit_has_the_keplerian_frequency():
    a, r0 = 0.9, 8.0
    d = math.sqrt(1 - 3 / r0 + 2 * a / r0 ** 1.5)
    E = (1 - 2 / r0 + a / r0 ** 1.5) / d                                   # Bardeen, Press & Teukolsky 1972
    L = math.sqrt(r0) * (1 - 2 * a / r0 ** 1.5 + a * a / r0 ** 2) / d
    st = [0.0, r0, math.pi / 2, 0.0, -E, 0.0, 0.0, L]
    s, status, _ = O.integrate_orbits(KERR, [st], dict(CFG, lambda_end=1000.0))
    assert status[0] == 0
    assert np.abs(s[0, :, 1] - r0).max() <= 1e-7
    assert s[0, -1, 3] / s[0, -1, 0] == pytest.approx(1.0 / (r0 ** 1.5 + a), rel=1e-9)   # Omega_K
    assert np.allclose(s[0, :, 6], -1.0, atol=1e-9)


def test_perihelion_precession_against_the_orbit_integral():
    """PAPER.md Fig 1 ("perihelion precession"): a bound eccentric Schwarzschild orbit; the advance of the
    periapsis per radial period from the sampled trajectory against 2 int_{r1}^{r2} dphi/dr dr."""
    E, L = 0.97, 4.2
    # turning points: E^2 = (1 - 2/r)(1 + L^2/r^2)
    roots = np.roots([E * E - 1, 2.0, -L * L, 2 * L * L])
    r1, r2 = sorted(x.real for x in roots if abs(x.imag) < 1e-12 and x.real > 5.0)
    f = lambda r: (L / r ** 2) / math.sqrt(max(E * E - (1 - 2 / r) * (1 + L * L / r ** 2), 1e-300))
    # substitute r = mid + half sin(x) to tame the inverse-square-root end points
    mid, half = 0.5 * (r1 + r2), 0.5 * (r2 - r1)
    dphi_exact = 2 * quad(lambda x: f(mid + half * math.sin(x)) * half * math.cos(x), -math.pi / 2, math.pi / 2,
                          epsabs=1e-13, epsrel=1e-13)[0]
    st = [0.0, r1, math.pi / 2, 0.0, -E, 0.0, 0.0, L]                       # start at periapsis
    K = 6000
    s, status, _ = O.integrate_orbits(SCHW, [st], dict(CFG, lambda_end=3000.0, n_samples=K, h_max=0.5))
    assert status[0] == 0
    lam, r, phi = s[0, :, 7], s[0, :, 1], s[0, :, 3]
    mins = [i for i in range(1, K - 1) if r[i] < r[i - 1] and r[i] <= r[i + 1]]
    assert len(mins) >= 2

    def vertex(i):      # parabola through three samples of r(lambda); phi interpolated at its vertex
        x, yv = lam[i - 1:i + 2], r[i - 1:i + 2]
        c = np.polyfit(x - x[1], yv, 2)
        xv = -c[1] / (2 * c[0])
        return np.polyval(np.polyfit(x - x[1], phi[i - 1:i + 2], 2), xv)
    adv = vertex(mins[1]) - vertex(mins[0])
    assert adv == pytest.approx(dphi_exact, rel=2e-6)
    assert dphi_exact > 2 * math.pi + 0.5                                   # a strong-field precession
    assert np.allclose(s[0, :, 6], -1.0, atol=1e-9)


def test_generic_kerr_timelike_orbit_against_scipy_dop853():
    st = np.array([0.0, 9.0, 1.2, 0.3, -0.95, 0.05, 1.5, 2.8])
    gi = O.metric_inv(KERR, st[1], st[2])[:5]
    # scale p_r so that 2H = -1 exactly at the start
    rest = gi[0] * st[4] ** 2 + 2 * gi[1] * st[4] * st[7] + gi[2] * st[7] ** 2 + gi[4] * st[6] ** 2
    st[5] = math.sqrt((-1.0 - rest) / gi[3])
    cfg = dict(CFG, lambda_end=400.0, n_samples=8)
    s, status, _ = O.integrate_orbits(KERR, [st], cfg)
    assert status[0] == 0

    def F(lam, y):
        full = np.array([y[0], y[1], y[2], y[3], st[4], y[4], y[5], st[7]])
        return O.rhs(KERR, full)
    sol = solve_ivp(F, (0.0, 400.0), [st[0], st[1], st[2], st[3], st[5], st[6]], method="DOP853", rtol=1e-13,
                    atol=1e-13, t_eval=s[0, :, 7])
    assert np.abs(sol.y.T - s[0, :, :6]).max() <= 2e-8
    assert np.allclose(s[0, :, 6], -1.0, atol=1e-8)


def test_plunging_orbit_ends_captured_and_leaves_nan_samples():
    E, L = 0.95, 3.0                                                        # below the marginally bound L = 4
    st = [0.0, 12.0, math.pi / 2, 0.0, -E, -0.1, 0.0, L]
    gi = O.metric_inv(SCHW, 12.0, math.pi / 2)[:5]
    st[5] = -math.sqrt((-1.0 - gi[0] * E * E - gi[2] * L * L) / gi[3])      # inward, 2H = -1
    s, status, _ = O.integrate_orbits(SCHW, [st], dict(CFG, lambda_end=500.0, n_samples=100))
    assert status[0] == 1
    done = ~np.isnan(s[0, :, 1])
    assert 0 < done.sum() < 100 and not done[done.argmin():].any()           # a prefix of samples, then NaN
    assert s[0, done, 1].min() > 2.0


def test_null_orbit_from_the_camera_keeps_H_zero():
    w = W.workload("C2")
    st = O.initial_state(w["metric"], w["camera"], 9.0, 2.0)
    s, status, _ = O.integrate_orbits(w["metric"], [st], dict(CFG, lambda_end=1500.0, h_max=100.0, h0=10.0))
    assert status[0] == 0
    assert np.abs(s[0, :, 6]).max() <= 1e-9
    assert s[0, :, 1].min() < 20.0 and s[0, -1, 1] > 400.0                    # went in and came back out
