"""Pins for the oracle's whole-trajectory output: closed forms, textbook quadratures, exact
classifiers, conserved quantities, symmetry, and an independent library integrator.
Citations: P:Lnnn = PAPER.md line; Rn = DESIGN.md section 3 reading.
"""
import copy
import math

import numpy as np
import pytest
from scipy.integrate import quad, solve_ivp
from scipy.optimize import brentq

import gp_workloads as W
from oracle import oracle as O

TWO_PI = 2 * math.pi


def angle_diff(a, b):
    return (a - b + math.pi) % TWO_PI - math.pi


# ---- P1: flat space (Schwarzschild with M = 0; the situation of Fig 6) ------------
def _flat_workload(scheme):
    w = W.workload("C1")
    w["metric"]["M"] = 0.0
    w["camera"].update(theta_obs=1.1, phi_obs=0.4)
    if scheme == 2:
        w["cfg"].update(scheme=2, rtol=1e-12, atol=1e-12, h_cap_rel=0.1, max_steps=100000)
    return w


@pytest.mark.parametrize("scheme,tol", [(2, 2e-10), (0, 1e-6)])
def test_flat_space_rays_are_straight_lines(scheme, tol):
    """Ray = x_o + lambda n with |n| = 1 (unit locally measured energy, R12/R13):
    exit lambda = r_o^2/D + sqrt(r_o^4/D^2 + r_esc^2 - r_o^2), t = -lambda (time-reversed trace),
    exit (theta, phi) from the Cartesian end point.  Pins the camera conventions
    (pinhole direction (-r_o, -beta, alpha)/D in the (r, theta, phi) frame), the landing step and
    the affine scale."""
    w = _flat_workload(scheme)
    ro, th0, ph0, resc = 50.0, 1.1, 0.4, 100.0
    er = np.array([math.sin(th0) * math.cos(ph0), math.sin(th0) * math.sin(ph0), math.cos(th0)])
    eth = np.array([math.cos(th0) * math.cos(ph0), math.cos(th0) * math.sin(ph0), -math.sin(th0)])
    eph = np.array([-math.sin(ph0), math.cos(ph0), 0.0])
    rays = ((3.0, -2.0), (-7.5, 0.5), (0.3, 9.0), (-9.9, -9.9), (1e-3, 2e-3))
    if scheme == 0:
        # fixed h = 0.05 cannot resolve a fly-by of the polar axis or of the origin in spherical
        # coordinates (1/sin^2(theta), 1/r^2 terms; P:L723 notes the same breakage): keep |alpha| >= 3
        rays = rays[:2] + rays[3:4]
    for al, be in rays:
        rec, _ = O.trace_one(w, al, be)
        D = math.sqrt(ro * ro + al * al + be * be)
        lam = ro * ro / D + math.sqrt(ro**4 / D**2 + resc**2 - ro**2)
        X = ro * er + lam * (-ro * er - be * eth + al * eph) / D
        assert rec["status"] == 0 and rec["r"] == resc
        assert rec["lambda"] == pytest.approx(lam, abs=tol * 100)
        assert rec["t"] == pytest.approx(-lam, abs=tol * 100)
        assert rec["theta"] == pytest.approx(math.acos(X[2] / resc), abs=tol)
        assert angle_diff(rec["phi"], math.atan2(X[1], X[0])) == pytest.approx(0.0, abs=tol)
        assert rec["p_t"] == pytest.approx(1.0, abs=1e-15)


# ---- P2: Schwarzschild ------------------------------------------------------------------
def _schw_adaptive():
    w = W.workload("C1")
    w["cfg"].update(scheme=2, rtol=1e-11, atol=1e-11, h_cap_rel=0.1, max_steps=100000)
    return w


def _impact(rec):
    """b = L/E from the record's constants at the observer on the equator (theta = pi/2):
    L^2 = p_theta^2 + p_phi^2/sin^2(theta)."""
    w = W.workload("C1")
    st = O.initial_state(w["metric"], w["camera"], rec["alpha"], rec["beta"])
    return math.hypot(st[6], st[7]) / st[4]


def test_schwarzschild_capture_iff_b_below_critical():
    """P:L139 + textbook: a photon from outside is captured iff b < 3 sqrt(3) M.  Also pins
    b = r_o sin(psi)/sqrt(1 - 2M/r_o) with tan(psi) = sqrt(alpha^2+beta^2)/r_o."""
    bc = 3 * math.sqrt(3)
    for wl, band in ((W.workload("C1"), 2e-2), (_schw_adaptive(), 1e-6)):
        rec, _ = O.trace(wl)
        b = np.array([_impact(r) for r in rec])
        psi = np.arctan(np.hypot(rec["alpha"], rec["beta"]) / 50.0)
        assert np.allclose(b, 50.0 * np.sin(psi) / math.sqrt(1 - 2 / 50.0), rtol=1e-13)
        sure = np.abs(b - bc) > band
        if wl["cfg"]["scheme"] == 0:  # fixed-step RK4 breaks down for rays grazing the polar axis
            sure &= rec["sin_theta_min"] > 0.05
        assert sure.sum() > 3000
        assert np.array_equal(rec["status"][sure] == 1, b[sure] < bc)
        assert set(np.unique(rec["status"][sure])) == {0, 1}
    # bisect the shadow edge along the alpha axis with the adaptive scheme
    wl = _schw_adaptive()
    edge = brentq(lambda a: O.trace_one(wl, a, 0.0)[0]["status"] - 0.5, 4.0, 6.0, xtol=1e-9)
    b_edge = 50.0 * math.sin(math.atan(edge / 50.0)) / math.sqrt(1 - 2 / 50.0)
    assert b_edge == pytest.approx(bc, abs=1e-6)


def _schw_quadratures(b, ro, resc):
    """Textbook orbit integrals for a photon with impact parameter b > b_c, E = 1:
    swept angle = int b dr / (r^2 sqrt(1 - b^2 F/r^2)), lambda = int dr / sqrt(1 - b^2 F/r^2),
    t = int dr / (F sqrt(...)), F = 1 - 2/r, over r_p -> r_o and r_p -> r_esc."""
    Veff = lambda r: 1 - b * b * (1 - 2 / r) / (r * r)
    rp = brentq(Veff, 3.0, b * 1.5)
    out = np.zeros(3)
    for rmax in (ro, resc):
        smax = math.sqrt(rmax - rp)
        for i, g in enumerate((lambda r: b / (r * r), lambda r: 1.0, lambda r: 1 / (1 - 2 / r))):
            # r = rp + s^2 removes the inverse-square-root end point singularity
            val, _ = quad(lambda s: g(rp + s * s) * 2 * s / math.sqrt(max(Veff(rp + s * s), 1e-300)),
                          0, smax, epsabs=1e-13, epsrel=1e-13, limit=400)
            out[i] += val
    return out


@pytest.mark.parametrize("al,be", [(7.0, 0.0), (5.5, 3.0), (-4.0, 8.0), (-5.3, -0.4)])
def test_schwarzschild_deflection_and_travel_time_quadrature(al, be):
    wl = _schw_adaptive()
    rec, _ = O.trace_one(wl, al, be)
    assert rec["status"] == 0
    E = rec["p_t"]
    b = _impact(rec)
    dpsi, lam, t = _schw_quadratures(b, 50.0, 100.0)
    # angle swept in the orbital plane between the observer direction and the exit direction
    cosw = math.sin(rec["theta"]) * math.cos(rec["phi"])  # observer at theta = pi/2, phi = 0
    assert cosw == pytest.approx(math.cos(dpsi), abs=2e-9)
    assert rec["lambda"] == pytest.approx(lam / E, rel=2e-10)  # dr/dlambda scales with E
    assert rec["t"] == pytest.approx(-t, rel=2e-10)


# ---- P3: Kerr shadow ------------------------------------------------------------------------
def _kerr_captured_exact(st, M, a, ro):
    """A null ray that starts inward at r_o falls through the horizon iff the radial potential
    R(r) = ((r^2+a^2) p_t + a p_phi)^2 - Delta (Q + (p_phi + a p_t)^2) has no zero in (r_+, r_o)
    (Carter 1968; covector form, so it is convention-free)."""
    pt, pth, pph = st[4], st[6], st[7]
    th = st[2]
    Q = pth**2 + math.cos(th) ** 2 * (pph**2 / math.sin(th) ** 2 - a * a * pt * pt)
    K = Q + (pph + a * pt) ** 2
    # quartic in r
    P = np.poly1d([pt, 0.0, a * a * pt + a * pph])
    R = P * P - np.poly1d([1.0, -2 * M, a * a]) * K
    rp = M + math.sqrt(M * M - a * a)
    roots = [z.real for z in R.roots if abs(z.imag) < 1e-9 * max(1.0, abs(z.real)) and rp < z.real < ro]
    return len(roots) == 0, R


def test_kerr_capture_matches_radial_potential_classifier():
    wl = W.workload("C2")
    rec, _ = O.trace(wl, ray_begin=3, ray_stride=101)
    assert set(np.unique(rec["status"])) == {0, 1}
    n_checked = 0
    for r in rec:
        st = O.initial_state(wl["metric"], wl["camera"], r["alpha"], r["beta"])
        cap, R = _kerr_captured_exact(st, 1.0, 0.9, 1000.0)
        # skip rays within 1e-6 of the shadow edge (double root of R)
        crit = [z.real for z in R.deriv().roots if abs(z.imag) < 1e-12 and z.real > 1.4359]
        if any(abs(R(c)) < 1e-6 * st[4] ** 2 * c**4 for c in crit):
            continue
        n_checked += 1
        assert (r["status"] == 1) == cap, (r["alpha"], r["beta"])
    assert n_checked > 2500 and (rec["status"] == 1).sum() > 200


def test_kerr_shadow_edges_against_bardeen_curve():
    """Bardeen (1973) critical curve for r_o -> infinity: xi_c(r), eta_c(r); on the image plane
    alpha = -xi/sin i, beta = +-sqrt(eta + a^2 cos^2 i - xi^2 cot^2 i).  At r_o = 1000 M the
    traced edge must agree to O(M/r_o)."""
    a, inc = 0.9, math.radians(60.0)
    xi = lambda r: -(r**3 - 3 * r**2 + a * a * r + a * a) / (a * (r - 1))
    eta = lambda r: -(r**3) * (r**3 - 6 * r**2 + 9 * r - 4 * a * a) / (a * a * (r - 1) ** 2)
    beta2 = lambda r: eta(r) + a * a * math.cos(inc) ** 2 - xi(r) ** 2 / math.tan(inc) ** 2
    r1 = brentq(beta2, 1.56, 2.4)
    r2 = brentq(beta2, 2.6, 3.9)
    edges = sorted([-xi(r1) / math.sin(inc), -xi(r2) / math.sin(inc)])
    assert edges == pytest.approx([-3.0959080, 6.5894090], abs=2e-6)
    wl = W.workload("C2")
    f = lambda al: O.trace_one(wl, al, 0.0)[0]["status"] - 0.5
    got = [brentq(f, -4.0, -2.0, xtol=1e-8), brentq(f, 5.5, 7.5, xtol=1e-8)]
    assert got[0] == pytest.approx(edges[0], abs=0.01) and got[1] == pytest.approx(edges[1], abs=0.01)
    # the same bisection with the observer 100x farther away converges to the closed form
    far = copy.deepcopy(wl)
    far["camera"]["r_obs"] = 1e5
    far["cfg"]["r_escape"] = 1.1e5
    g = lambda al: O.trace_one(far, al, 0.0)[0]["status"] - 0.5
    got_far = [brentq(g, -4.0, -2.0, xtol=1e-8), brentq(g, 5.5, 7.5, xtol=1e-8)]
    assert got_far == pytest.approx(edges, abs=2e-4)
    # top of the shadow: beta_max = 5.1354684 at alpha = 1.5971344 (maximum of beta(r) on the curve)
    rr = np.linspace(r1, r2, 20001)
    bb = np.sqrt(np.maximum([beta2(r) for r in rr], 0))
    i = bb.argmax()
    assert bb[i] == pytest.approx(5.1354684, abs=1e-6)
    al_top = -xi(rr[i]) / math.sin(inc)
    hfar = lambda be: O.trace_one(far, al_top, be)[0]["status"] - 0.5
    assert brentq(hfar, 4.0, 6.5, xtol=1e-8) == pytest.approx(bb[i], abs=2e-4)


# ---- P4: invariants ---------------------------------------------------------------------
def test_kerr_invariants_on_config2_sample():
    """BASELINE.json: |H| drift <= 1e-8; Carter Q conserved.  On escaped rays; for
    captured rays |H| inflates at the coordinate singularity of the horizon (R22)."""
    rec, _ = O.trace(W.workload("C2"), ray_begin=11, ray_stride=257)
    esc = rec["status"] == 0
    assert esc.sum() > 800
    assert rec["h_max"][esc].max() < 1e-8
    assert rec["q_drift"][esc].max() < 1e-8
    assert rec["h_max"][~esc].max() < 1e-4
    # E and L_z are carried, not integrated: exact (R12)
    wl = W.workload("C2")
    for r in rec[:20]:
        st = O.initial_state(wl["metric"], wl["camera"], r["alpha"], r["beta"])
        assert r["p_t"] == st[4] and r["p_phi"] == st[7]
    # exit surface reached exactly, affine time ~ path length
    assert np.all(rec["r"][esc] == 1100.0)
    assert np.all(rec["r"][~esc] == O.radii(wl["metric"])[0] * (1 + 1e-3))
    assert np.all((rec["lambda"][esc] > 2090) & (rec["lambda"][esc] < 2200))


def test_step_accounting():
    wl = W.workload("C2")
    rec, _ = O.trace(wl, ray_begin=5, ray_stride=1001)
    assert np.all(rec["n_rhs"] == 1 + 6 * (rec["n_accepted"] + rec["n_rejected"]) + 5)
    assert 250 < rec["n_accepted"].mean() < 450 and rec["n_rejected"].mean() < 20
    wl = W.workload("C1")
    rec, _ = O.trace(wl, ray_stride=7)
    assert np.all(rec["n_rejected"] == 0)
    assert np.all(rec["n_rhs"] == 4 * rec["n_accepted"] + 3 * (rec["status"] < 2))
    assert np.all(np.isinf(rec["err_margin"]))
    # budget: attempted steps <= max_steps, status MAXSTEPS, record = current state (R18)
    wl["cfg"]["max_steps"] = 100
    rec, _ = O.trace(wl, ray_stride=7)
    assert np.all(rec["status"] == 2) and np.all(rec["n_accepted"] == 100)
    assert np.allclose(rec["lambda"], 100 * 0.05)


# ---- P14 / P5: limits ---------------------------------------------------------------------
def test_kerr_zero_spin_reproduces_schwarzschild_records():
    ws = _schw_adaptive()
    wk = copy.deepcopy(ws)
    wk["metric"].update(id=1, a=1e-13)
    rs, _ = O.trace(ws, ray_stride=13)
    rk, _ = O.trace(wk, ray_stride=13)
    assert np.array_equal(rs["status"], rk["status"])
    ok = rs["err_margin"] > 1e-6
    for f in ("theta", "phi", "lambda", "t"):
        assert np.allclose(rs[f][ok], rk[f][ok], rtol=0, atol=1e-9)


def test_manko_novikov_q0_reproduces_kerr_records():
    """BASELINE.json: 'q = 0 must reproduce Kerr'."""
    wk = W.workload("C2")
    wm = copy.deepcopy(wk)
    wm["metric"].update(id=2, q=0.0)
    rk, _ = O.trace(wk, ray_begin=17, ray_count=160, ray_stride=1601)
    rm, _ = O.trace(wm, ray_begin=17, ray_count=160, ray_stride=1601)
    assert np.array_equal(rk["status"], rm["status"])
    ok = (rk["err_margin"] > 1e-6) & (rk["n_accepted"] == rm["n_accepted"])
    assert ok.sum() > 150
    for f in ("theta", "phi", "lambda", "t"):
        assert np.allclose(rk[f][ok], rm[f][ok], rtol=0, atol=2e-11 * 2200)


# ---- P8: equatorial mirror symmetry of the Manko-Novikov image (Fig 4) --------------
def test_manko_novikov_image_is_mirror_symmetric_at_90_degrees():
    wl = W.workload("C4")
    n = 0
    for al, be in ((7.5, 2.0), (-7.0, 3.3), (9.0, 8.0), (-4.9, 5.2), (3.7, 7.1), (12.0, 0.7)):
        up, _ = O.trace_one(wl, al, be)
        dn, _ = O.trace_one(wl, al, -be)
        assert up["status"] == dn["status"] == 0
        if min(up["err_margin"], dn["err_margin"]) < 1e-6:
            continue
        n += 1
        assert up["theta"] + dn["theta"] == pytest.approx(math.pi, abs=1e-9)
        assert up["phi"] == pytest.approx(dn["phi"], abs=1e-9)
        assert up["lambda"] == pytest.approx(dn["lambda"], abs=1e-8)
        assert up["h_max"] < 1e-8
    assert n >= 4


def test_manko_novikov_shadow_is_taller_for_prolate_q():
    """P:L232, P:L426 (Fig 7): seen with the rotation axis vertical, the shadow gets taller for
    q < 0 (prolate) and less tall for q > 0 (oblate); shadow = rays that never leave.
    Equatorial observer, so the height is twice the upper edge on the column alpha = 2."""
    top = {}
    for q in (-0.5, 0.0, 0.5):
        wl = W.workload("C4")
        wl["metric"]["q"] = q
        wl["cfg"]["max_steps"] = 2000
        f = lambda be: (O.trace_one(wl, 2.0, be)[0]["status"] == 0) - 0.5
        top[q] = brentq(f, 4.0, 7.0, xtol=1e-4)
    assert top[-0.5] > top[0.0] + 0.05 and top[0.0] > top[0.5] + 0.05


# ---- P9 / P12: independent library integration of the same equations -----------------------
def _dop853_exit(wl, al, be, r_target, equator_events=False):
    m, cam = wl["metric"], wl["camera"]
    st = O.initial_state(m, cam, al, be)

    def f(_, y):
        return O.rhs(m, [y[0], y[1], y[2], y[3], st[4], y[4], y[5], st[7]])
    hit = lambda _, y: y[1] - r_target
    hit.terminal = True
    events = [hit]
    if equator_events:
        eq = lambda _, y: y[2] - math.pi / 2
        events.append(eq)
    sol = solve_ivp(f, (0, 1e5), [st[0], st[1], st[2], st[3], st[5], st[6]], method="DOP853",
                    rtol=1e-13, atol=1e-13, events=events, max_step=50.0)
    assert sol.status == 1
    return sol


@pytest.mark.parametrize("al,be", [(8.0, 1.0), (-6.0, 4.5), (2.0, -9.0), (-11.0, -11.0), (7.2, 0.3)])
def test_kerr_exit_state_against_scipy_dop853(al, be):
    """Truth by a different integrator (8th order, rtol 1e-13): at rtol 1e-10 the method's own
    truncation error on smooth rays is ~1e-10..1e-8."""
    wl = W.workload("C2")
    rec, _ = O.trace_one(wl, al, be)
    assert rec["status"] == 0
    sol = _dop853_exit(wl, al, be, 1100.0)
    y = sol.y_events[0][0]
    assert rec["theta"] == pytest.approx(y[2], abs=2e-8)
    assert rec["phi"] == pytest.approx(y[3], abs=2e-8)
    assert rec["lambda"] == pytest.approx(sol.t_events[0][0], abs=2e-6)
    assert rec["t"] == pytest.approx(y[0], abs=2e-6)
    assert rec["p_r"] == pytest.approx(y[4], abs=1e-9) and rec["p_theta"] == pytest.approx(y[5], abs=2e-6)


def test_manko_novikov_exit_state_against_scipy_dop853():
    wl = W.workload("C4")
    for al, be in ((8.0, 3.0), (-9.0, -2.5)):
        rec, _ = O.trace_one(wl, al, be)
        sol = _dop853_exit(wl, al, be, 1100.0)
        y = sol.y_events[0][0]
        assert rec["status"] == 0
        assert rec["theta"] == pytest.approx(y[2], abs=5e-8) and rec["phi"] == pytest.approx(y[3], abs=5e-8)
        assert rec["lambda"] == pytest.approx(sol.t_events[0][0], abs=5e-6)


def test_captured_ray_against_scipy_dop853():
    wl = W.workload("C2")
    rcap = O.radii(wl["metric"])[0] * (1 + 1e-3)
    rec, _ = O.trace_one(wl, 1.0, 0.5)
    assert rec["status"] == 1 and rec["r"] == rcap
    sol = _dop853_exit(wl, 1.0, 0.5, rcap)
    y = sol.y_events[0][0]
    assert rec["theta"] == pytest.approx(y[2], abs=1e-7)
    assert rec["lambda"] == pytest.approx(sol.t_events[0][0], abs=1e-6)


# ---- P13: disk crossings and redshift (config 3) ------------------------------------------------
def test_disk_crossings_against_event_location_and_g_sign():
    """R19: crossings of theta = pi/2 located by the landing step; only r_ISCO <= r <= 20 kept,
    in order along the traced ray; g from P:L372 (eq 57).  Truth: DOP853 event location."""
    wl = W.workload("C3")
    risco = O.radii(wl["metric"])[1]
    seen = 0
    for al, be in ((-8.0, 1.0), (8.0, 1.0), (3.0, -2.5), (-12.0, 3.0), (15.0, -1.0)):
        rec, _ = O.trace_one(wl, al, be)
        rt = 1100.0 if rec["status"] == 0 else O.radii(wl["metric"])[0] * (1 + 1e-3)
        sol = _dop853_exit(wl, al, be, rt, equator_events=True)
        rc_all = [y[1] for y in sol.y_events[1]]
        assert rec["n_equator_crossings"] == len(rc_all)
        want = [r for r in rc_all if risco <= r <= 20.0][:3]
        assert rec["n_disk_recorded"] == len(want)
        for i, r in enumerate(want):
            assert rec["disk_r"][i] == pytest.approx(r, abs=2e-8)
            g = O.kepler(wl["metric"], r, rec["p_t"], rec["p_phi"])[2]
            assert rec["disk_g"][i] == pytest.approx(g, rel=1e-7)
            seen += 1
        assert np.all(np.isnan(rec["disk_r"][len(want):]))
    assert seen >= 5
    # approaching (prograde, alpha < 0) side is blueshifted relative to the receding side (Fig 15)
    left, _ = O.trace_one(wl, -8.0, 1.0)
    right, _ = O.trace_one(wl, 8.0, 1.0)
    assert left["disk_g"][0] > 1.0 > right["disk_g"][0]


def test_disk_off_leaves_integration_untouched():
    w3 = W.workload("C3")
    w0 = copy.deepcopy(w3)
    w0["cfg"]["max_crossings"] = 0
    a, _ = O.trace(w3, ray_begin=9, ray_count=64, ray_stride=16001)
    b, _ = O.trace(w0, ray_begin=9, ray_count=64, ray_stride=16001)
    for f in ("status", "theta", "phi", "lambda", "n_accepted", "n_rejected", "n_equator_crossings"):
        assert np.array_equal(a[f], b[f])
    assert np.all(b["n_disk_recorded"] == 0) and a["n_disk_recorded"].sum() > 0


# ---- RK4 with h = h_rel r (config 5) converges to the adaptive result ------------------------------
def test_rk4_relative_step_converges_with_fourth_order():
    wl = W.workload("C5a")
    ref = W.workload("C5a")
    ref["cfg"].update(scheme=2, rtol=1e-12, atol=1e-12, h_cap_rel=0.1, max_steps=10**6)
    al, be = 9.0, 6.0
    truth, _ = O.trace_one(ref, al, be)
    errs = []
    for hrel in (0.04, 0.02, 0.01):
        wl["cfg"]["h_rel"] = hrel
        rec, _ = O.trace_one(wl, al, be)
        errs.append(abs(rec["phi"] - truth["phi"]) + abs(rec["theta"] - truth["theta"]))
    assert errs[1] < 1e-6
    assert 3.5 < math.log2(errs[0] / errs[1]) < 4.6 and 3.5 < math.log2(errs[1] / errs[2]) < 4.6
