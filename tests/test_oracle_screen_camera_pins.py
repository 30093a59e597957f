"""Pins of the oracle's Euclidean-screen camera (the paper's own, eq 51-55),
`projection = 1`.  CPU only."""
import copy
import math

import numpy as np
import pytest

import gp_workloads as W
from oracle import oracle as O

KERR = dict(id=W.KERR, M=1.0, a=0.9, q=0.0)
MN = dict(id=W.MANKO_NOVIKOV, M=1.0, a=0.9, q=0.5)
SCHW = dict(id=W.SCHWARZSCHILD, M=1.0, a=0.0, q=0.0)


def cam(theta_deg=60.0, phi=0.3, k2=0.0, r_obs=1000.0):
    c = copy.deepcopy(W.workload("C2")["camera"])
    c.update(projection=1, focal_2f_over_d=k2, theta_obs=math.radians(theta_deg), phi_obs=phi, r_obs=r_obs)
    return c


def bl_to_cart(a, r, th, ph):
    R = math.sqrt(r * r + a * a)                       # eq 51-53
    return np.array([R * math.sin(th) * math.cos(ph), R * math.sin(th) * math.sin(ph), r * math.cos(th)])


def frame(c):
    so, co, sp, cp = math.sin(c["theta_obs"]), math.cos(c["theta_obs"]), math.sin(c["phi_obs"]), math.cos(c["phi_obs"])
    return np.array([so * cp, so * sp, co]), np.array([-sp, cp, 0.0]), np.array([-co * cp, -co * sp, so])


@pytest.mark.parametrize("m", [SCHW, KERR, MN], ids=["schw", "kerr", "mn"])
@pytest.mark.parametrize("k2", [0.0, 0.02])
def test_start_point_is_on_the_screen_and_momentum_is_null_with_dt_minus_one(m, k2):
    c = cam(k2=k2)
    chat, eph, eup = frame(c)
    a = 0.0 if m["id"] == W.SCHWARZSCHILD else m["a"]
    for al, be in ((0.0, 0.0), (7.0, -3.0), (-11.5, 11.9), (2.5, 9.0)):
        st = O.initial_state(m, c, al, be)
        # eq 51-53 map the start point back onto the flat screen
        X = bl_to_cart(a, st[1], st[2], st[3])
        assert np.allclose(X, c["r_obs"] * chat + al * eph + be * eup, rtol=0, atol=1e-9)
        assert st[0] == 0.0
        # null (eq 54) and dt/dlambda = -1, from the inverse metric the tracer integrates
        gi = O.metric_inv(m, st[1], st[2])[:5]
        gtt, gtp, gpp, grr, gthth = gi
        pt, pr, pth, pph = st[4], st[5], st[6], st[7]
        H2 = gtt * pt * pt + 2 * gtp * pt * pph + gpp * pph * pph + grr * pr * pr + gthth * pth * pth
        assert abs(H2) <= 1e-12
        assert gtt * pt + gtp * pph == pytest.approx(-1.0, abs=1e-12)
        # the contravariant direction, pushed forward with the Jacobian of eq 51-53 by finite
        # differences, is the Euclidean direction -c_hat + k2 (alpha e_phi + beta e_up) up to scale
        qdot = np.array([grr * pr, gthth * pth, gtp * pt + gpp * pph])      # (dr, dtheta, dphi)/dlambda
        J = np.zeros((3, 3))
        for k in range(3):
            h = 1e-6 * (st[1] if k == 0 else 1.0)
            p, q = st[1:4].copy(), st[1:4].copy()
            p[k] += h
            q[k] -= h
            J[:, k] = (bl_to_cart(a, *p) - bl_to_cart(a, *q)) / (2 * h)
        v = J @ qdot
        want = -chat + k2 * (al * eph + be * eup)
        assert np.allclose(v / np.linalg.norm(v), want / np.linalg.norm(want), atol=2e-8)


def test_flat_space_parallel_rays_all_leave_in_the_same_direction():
    """M = 0: straight lines.  Parallel rays (focal distance infinity) all exit towards -c_hat; the
    exit time follows from the chord.  (The ray through the screen centre runs through r = 0, where the
    spherical chart is singular, so it is left out.)"""
    w = W.workload("C1")
    w["metric"]["M"] = 0.0
    w["camera"].update(projection=1, focal_2f_over_d=0.0, theta_obs=1.1, phi_obs=0.4)
    w["cfg"].update(scheme=2, rtol=1e-12, atol=1e-12, h_cap_rel=0.1, max_steps=100000)
    chat, eph, eup = frame(w["camera"])
    for al, be in ((1.0, 0.5), (6.0, 2.0), (-9.0, -9.5)):
        rec, _ = O.trace_one(w, al, be)
        assert rec["status"] == 0
        X0 = 50.0 * chat + al * eph + be * eup
        # straight line X0 - s c_hat leaves the sphere r = 100 at s = X0.c_hat + sqrt(100^2 - |X0_perp|^2)
        perp2 = al * al + be * be
        s = 50.0 + math.sqrt(100.0 ** 2 - perp2)
        Xe = X0 - s * chat
        assert math.cos(rec["theta"]) == pytest.approx(Xe[2] / 100.0, abs=1e-10)
        dphi = (rec["phi"] - math.atan2(Xe[1], Xe[0]) + math.pi) % (2 * math.pi) - math.pi
        assert abs(dphi) <= 1e-10
        assert rec["lambda"] == pytest.approx(s, rel=1e-10)      # dt/dlambda = -1 and |dX/dlambda| = 1
        assert rec["t"] == pytest.approx(-s, rel=1e-10)


def test_kerr_shadow_edges_seen_with_parallel_rays_are_bardeens():
    """Parallel rays from a far screen carry impact parameters (alpha, beta) = screen coordinates, so
    the shadow edge on the beta = 0 line sits at Bardeen's alpha = -3.0959080 and +6.5894090
    (a = 0.9, i = 60 deg; SURVEY.md pin P3), up to the O(M/r_obs) correction of a screen at r = 1000."""
    w = W.workload("C2")
    w["camera"].update(projection=1, focal_2f_over_d=0.0)

    def captured(al):
        rec, _ = O.trace_one(w, al, 0.0)
        return rec["status"] == 1

    for lo, hi, edge in ((-3.6, -2.6, -3.0959080), (6.0, 7.2, 6.5894090)):
        a, b = lo, hi
        assert captured(a) != captured(b)
        for _ in range(40):
            mid = 0.5 * (a + b)
            if captured(mid) == captured(a):
                a = mid
            else:
                b = mid
        assert 0.5 * (a + b) == pytest.approx(edge, abs=0.02)


def test_mn_equatorial_screen_image_is_mirror_symmetric():
    w = W.workload("C4")
    w["camera"].update(projection=1, focal_2f_over_d=0.0)
    w["cfg"]["max_steps"] = 3000
    for al, be in ((8.0, 3.0), (-9.5, 6.0), (12.0, 11.0)):
        up, _ = O.trace_one(w, al, be)
        dn, _ = O.trace_one(w, al, -be)
        assert up["status"] == dn["status"] == 0
        assert up["theta"] + dn["theta"] == pytest.approx(math.pi, abs=1e-8)
        assert up["phi"] == pytest.approx(dn["phi"], abs=1e-8)
        assert up["lambda"] == pytest.approx(dn["lambda"], rel=1e-9)


def test_perspective_factor_widens_the_field_of_view():
    """With 2f/d > 0 the ray through (alpha, 0) leaves the screen tilted by atan(2f/d alpha): in flat
    space its exit direction is that Euclidean direction."""
    w = W.workload("C1")
    w["metric"]["M"] = 0.0
    w["camera"].update(projection=1, focal_2f_over_d=0.05, theta_obs=math.pi / 2, phi_obs=0.0)
    w["cfg"].update(scheme=2, rtol=1e-12, atol=1e-12, h_cap_rel=0.1, max_steps=100000)
    chat, eph, eup = frame(w["camera"])
    al = 8.0
    rec, _ = O.trace_one(w, al, 0.0)
    X0 = 50.0 * chat + al * eph
    V = -chat + 0.05 * al * eph
    V /= np.linalg.norm(V)
    b = X0 @ V
    s = -b + math.sqrt(b * b - (X0 @ X0) + 100.0 ** 2)
    Xe = X0 + s * V
    assert math.cos(rec["theta"]) == pytest.approx(Xe[2] / 100.0, abs=1e-10)
    dphi = (rec["phi"] - math.atan2(Xe[1], Xe[0]) + math.pi) % (2 * math.pi) - math.pi
    assert abs(dphi) <= 1e-10
