"""Pins of the oracle's solid-ring object (PAPER.md L444, L735 Figs 15-17; reading R39;
SURVEY.md section 8(f) NEXT-4, second half).

The ring is the volume r_in <= r <= r_out, |theta - pi/2| <= d; a ray ends on the face it enters
through (status 5), located by a landing step.  What fixes that other than the oracle itself:
  * flat space (M = 0): the ray is a straight line, the entry point into the volume is found here by
    dense sampling and bisection of the line, independently of any integrator;
  * thin limit d -> 0: the hit is the first equator crossing inside [r_in, r_out], which the thin-disk
    machinery (pinned by tests/test_oracle_trace_pins.py against event location) already records;
  * reflection symmetry about the equator for an equatorial observer (Kerr and Manko-Novikov);
  * every hit lies exactly on a face of the volume and inside the other coordinate's range.
"""
import copy
import math

import numpy as np
import pytest

import gp_workloads as W
from oracle import oracle as O


def ring_workload(name="C3", d=0.05, r_in=6.0, r_out=14.0, **cam):
    w = W.workload(name, **cam)
    w["cfg"].update(max_crossings=0, disk_r_in=r_in, disk_r_out=r_out, ring_half_angle=d)
    return w


def test_flat_space_entry_point_by_brute_force():
    w = ring_workload("C1", d=0.08, r_in=8.0, r_out=30.0, width=16, height=16, jitter_amp_px=0.0,
                      theta_obs=1.25, phi_obs=0.3, alpha_min=-32.0, alpha_max=32.0, beta_min=-32.0, beta_max=32.0)
    w["metric"]["M"] = 0.0
    w["cfg"].update(scheme=2, rtol=1e-12, atol=1e-12, h_cap_rel=0.1, max_steps=100000)
    rec, _ = O.trace(w)
    ab = O.alpha_beta(w["camera"], np.arange(len(rec)))
    ro, th0, ph0, d, r_in, r_out = 50.0, 1.25, 0.3, 0.08, 8.0, 30.0
    er = np.array([math.sin(th0) * math.cos(ph0), math.sin(th0) * math.sin(ph0), math.cos(th0)])
    eth = np.array([math.cos(th0) * math.cos(ph0), math.cos(th0) * math.sin(ph0), -math.sin(th0)])
    eph = np.array([-math.sin(ph0), math.cos(ph0), 0.0])

    def inside(X):
        r = np.linalg.norm(X)
        return r_in <= r <= r_out and abs(math.acos(X[2] / r) - math.pi / 2) <= d
    hits = 0
    for k in range(len(rec)):
        a, b = ab[k]
        D = math.sqrt(ro * ro + a * a + b * b)
        n = (-ro * er - b * eth + a * eph) / D
        X = lambda lam: ro * er + lam * n
        lam_hit = None
        lams = np.linspace(0.0, 160.0, 64001)
        flags = np.array([inside(X(l)) for l in lams[::8]])
        if flags.any():
            i = int(np.argmax(flags)) * 8
            lo, hi = lams[max(i - 8, 0)], lams[i]
            # refine the first entry: scan the bracketing interval finely, then bisect
            fine = np.linspace(lo, hi, 4001)
            j = int(np.argmax([inside(X(l)) for l in fine]))
            lo, hi = fine[max(j - 1, 0)], fine[j]
            for _ in range(80):
                mid = 0.5 * (lo + hi)
                lo, hi = (lo, mid) if inside(X(mid)) else (mid, hi)
            lam_hit = hi
        if lam_hit is None:
            assert rec["status"][k] == 0, (k, a, b)
            continue
        hits += 1
        assert rec["status"][k] == 5, (k, a, b, lam_hit)
        P = X(lam_hit)
        r = np.linalg.norm(P)
        assert abs(rec["lambda"][k] - lam_hit) <= 1e-8 and abs(rec["t"][k] + lam_hit) <= 1e-8
        assert abs(rec["r"][k] - r) <= 1e-8 and abs(rec["theta"][k] - math.acos(P[2] / r)) <= 1e-9
        dphi = (rec["phi"][k] - math.atan2(P[1], P[0]) + math.pi) % (2 * math.pi) - math.pi
        assert abs(dphi) <= 1e-9
        assert rec["disk_r"][k, 0] == rec["r"][k]
    on_theta_face = np.isclose(np.abs(rec["theta"] - math.pi / 2), d, rtol=0, atol=1e-15) & (rec["status"] == 5)
    on_r_face = (rec["r"] == r_out) & (rec["status"] == 5)
    assert hits > 20 and on_theta_face.sum() > 10 and on_r_face.sum() >= 2    # both kinds of face are exercised


@pytest.mark.parametrize("name", ["C3"])
def test_thin_limit_is_the_first_disk_crossing(name):
    """d -> 0: the ring hit is the first equator crossing with r_in <= r <= r_out, which the thin-disk path
    records as disk_r[0], with the same redshift factor; rays the disk never records are untouched."""
    thin = W.workload(name)
    thin["cfg"].update(disk_r_in=6.0, disk_r_out=14.0)
    ring = ring_workload(name, d=1e-11)
    sel = W.ray_selection(thin, 5, None, 523)
    a, _ = O.trace(thin, *sel)
    b, _ = O.trace(ring, *sel)
    hit = a["n_disk_recorded"] >= 1
    assert hit.sum() > 50 and (~hit).sum() > 500
    assert (b["status"][hit] == 5).all() and (b["status"][~hit] == a["status"][~hit]).all()
    assert np.abs(b["disk_r"][hit, 0] - a["disk_r"][hit, 0]).max() <= 1e-8     # the face is 1e-11 rad off the equator, dr/dtheta <= 1e2
    assert np.abs(b["disk_g"][hit, 0] / a["disk_g"][hit, 0] - 1.0).max() <= 1e-8
    for f in ("theta", "phi", "lambda", "t"):
        assert np.allclose(b[f][~hit], a[f][~hit], rtol=0, atol=0)               # same arithmetic, same bits


@pytest.mark.parametrize("metric,r_in", [(dict(id=W.KERR, M=1.0, a=0.98, q=0.0), 4.0),
                                         (dict(id=W.MANKO_NOVIKOV, M=1.0, a=0.1, q=-2.0), 5.0)])
def test_mirror_symmetry_for_an_equatorial_observer(metric, r_in):
    """PAPER.md Figs 15-17 configurations (a = 0.98 M Kerr; Manko-Novikov a = 0.1 M, q = -2) seen from the
    equator: the image of the ring is mirror-symmetric, (alpha, beta) <-> (alpha, -beta)."""
    w = ring_workload("C3", d=0.06, r_in=r_in, r_out=12.0, width=48, height=48, theta_obs=math.pi / 2,
                      alpha_min=-16.0, alpha_max=16.0, beta_min=-16.0, beta_max=16.0)
    w["metric"] = metric
    w["cfg"]["max_steps"] = 4000
    rec, _ = O.trace(w)
    img = rec.reshape(48, 48)
    up, dn = img[24:, :], img[:24, :][::-1, :]
    assert (up["status"] == dn["status"]).mean() >= 0.995
    ok = (up["status"] == 5) & (dn["status"] == 5) & (up["n_accepted"] < 600) & (dn["n_accepted"] < 600)
    assert ok.sum() > 100
    assert np.abs(up["r"] - dn["r"])[ok].max() <= 1e-7
    assert np.abs(up["theta"] + dn["theta"] - math.pi)[ok].max() <= 1e-8
    assert np.abs(up["disk_g"][..., 0] / dn["disk_g"][..., 0] - 1.0)[ok].max() <= 1e-7
    g = up["disk_g"][..., 0][ok]
    assert (g > 1.0).any() and (g < 1.0).any()       # approaching and receding sides (red / blue)


def test_hits_lie_on_a_face_of_the_volume():
    d, r_in, r_out = 0.05, 6.0, 14.0
    w = ring_workload("C3", d=d, r_in=r_in, r_out=r_out)
    rec, _ = O.trace(w, 3, None, 331)
    h = rec[rec["status"] == 5]
    assert len(h) > 150
    on_th = np.abs(np.abs(h["theta"] - math.pi / 2) - d) <= 1e-15
    on_r = (h["r"] == r_in) | (h["r"] == r_out)
    assert (on_th | on_r).all() and on_th.sum() > 100 and on_r.sum() >= 5
    assert ((h["r"] >= r_in) & (h["r"] <= r_out)).all()
    assert (np.abs(h["theta"] - math.pi / 2) <= d + 1e-15).all()
    assert np.array_equal(h["disk_r"][:, 0], h["r"]) and np.isfinite(h["disk_g"][:, 0]).all()
    assert (h["n_disk_recorded"] == 1).all()
    # the observer sits above the equator (80 degrees): the direct image is the top face
    assert (h["theta"][on_th] < math.pi / 2).mean() > 0.6
    # |H| stays at rounding level up to the hit
    assert np.percentile(h["h_max"], 99) <= 1e-9


def test_ring_validation():
    w = ring_workload("C3")
    w["cfg"]["max_crossings"] = 3
    with pytest.raises(ValueError):
        O.trace(w, 0, 4, 1)
    w = ring_workload("C3", r_in=9.0, r_out=8.0)      # empty radial range
    with pytest.raises(ValueError):
        O.trace(w, 0, 4, 1)


def test_ring_with_the_fixed_step_scheme_converges_to_the_adaptive_hits():
    """The ring with RK4 h = 0.01 r: same landing rule with the scheme's own step formula (R14).  The hit
    points agree with the adaptive scheme's to the fixed step's own accuracy, and every hit is on a face."""
    w2 = ring_workload("C3", d=0.05, r_in=6.0, r_out=14.0)
    w1 = copy.deepcopy(w2)
    w1["cfg"].update(scheme=1, h_rel=0.01, max_steps=200000)
    sel = W.ray_selection(w2, 7, None, 877)
    a, _ = O.trace(w2, *sel)
    b, _ = O.trace(w1, *sel)
    both = (a["status"] == 5) & (b["status"] == 5)
    assert both.sum() > 60 and (a["status"] == b["status"]).mean() > 0.99
    same_face = np.isclose(np.abs(a["theta"] - math.pi / 2), 0.05, atol=1e-15) == np.isclose(np.abs(b["theta"] - math.pi / 2), 0.05, atol=1e-15)
    ok = both & same_face
    assert ok.sum() >= 0.97 * both.sum()
    assert np.abs(a["r"] - b["r"])[ok].max() <= 1e-5 and np.abs(a["phi"] - b["phi"])[ok].max() <= 1e-5
    assert np.abs(a["disk_g"][ok, 0] / b["disk_g"][ok, 0] - 1.0).max() <= 1e-5
    on_face = np.isclose(np.abs(b["theta"][both] - math.pi / 2), 0.05, atol=1e-15) | (b["r"][both] == 6.0) | (b["r"][both] == 14.0)
    assert on_face.all()
