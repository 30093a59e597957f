"""Pins of the general-metric disk emitter (eq 56 solved with the metric's own derivatives; PAPER.md
L358-370, L372-374 eq 57; Figs 15-17).  CPU only."""
import math

import numpy as np
import pytest

import gp_workloads as W
from oracle import oracle as O

KERR = dict(id=W.KERR, M=1.0, a=0.9, q=0.0)
KERR_RETRO = dict(id=W.KERR, M=1.0, a=-0.6, q=0.0)
SCHW = dict(id=W.SCHWARZSCHILD, M=1.0, a=0.0, q=0.0)
MN0 = dict(id=W.MANKO_NOVIKOV, M=1.0, a=0.9, q=0.0)
MN = dict(id=W.MANKO_NOVIKOV, M=1.0, a=0.9, q=0.5)
MNP = dict(id=W.MANKO_NOVIKOV, M=1.0, a=0.1, q=-2.0)        # the paper's Fig 17 ring: a = 0.1 M, q = -2


@pytest.mark.parametrize("m", [SCHW, KERR, KERR_RETRO], ids=["schw", "kerr", "kerr_retro"])
def test_eq56_solve_reproduces_the_closed_form_keplerian_emitter(m):
    for r in (3.5 if m["a"] > 0 else 7.0, 6.0, 11.0, 40.0):
        for pt, pph in ((1.0, -3.0), (0.98, 5.5)):
            closed = O.kepler(m, r, pt, pph)
            solved = O.kepler_general(m, r, pt, pph)
            assert np.allclose(solved, closed, rtol=1e-11), (r, solved, closed)
    # spot value of SURVEY.md pin P11: a = 0.998, r = 6: Omega_K = 0.06371480861546, u^t = 1.33927221892028
    sv = O.kepler_general(dict(id=W.KERR, M=1.0, a=0.998, q=0.0), 6.0, 1.0, 0.0)
    assert sv[0] == pytest.approx(0.06371480861546, rel=1e-11)
    assert sv[1] == pytest.approx(1.33927221892028, rel=1e-11)


def test_manko_novikov_at_q0_has_the_kerr_emitter():
    for r in (4.0, 9.0, 25.0):
        assert np.allclose(O.kepler_general(MN0, r, 1.0, -2.0), O.kepler(KERR, r, 1.0, -2.0), rtol=1e-9)


@pytest.mark.parametrize("m", [MN, MNP], ids=["q0.5", "q-2"])
def test_the_emitter_of_eq56_is_a_circular_geodesic_of_the_manko_novikov_spacetime(m):
    """Dynamic pin: the covector that eq 56 gives, normalised to p^2 = -1, is handed to the orbit
    integrator; the orbit must stay on its circle and turn with the angular velocity eq 56 predicted."""
    for r0 in (7.0, 12.0):
        Om, ut, _ = O.kepler_general(m, r0, 1.0, 0.0)
        gi = O.metric_inv(m, r0, math.pi / 2)[:5]
        # u_mu = (u_t, 0, 0, u_phi) from u^t, u^phi = Omega u^t:  solve g^{t mu}u_mu = u^t, g^{phi mu}u_mu = Omega u^t
        A = np.array([[gi[0], gi[1]], [gi[1], gi[2]]])
        u_t, u_ph = np.linalg.solve(A, [ut, Om * ut])
        assert gi[0] * u_t ** 2 + 2 * gi[1] * u_t * u_ph + gi[2] * u_ph ** 2 == pytest.approx(-1.0, abs=1e-12)
        st = [0.0, r0, math.pi / 2, 0.0, u_t, 0.0, 0.0, u_ph]
        s, status, _ = O.integrate_orbits(m, [st], dict(rtol=1e-11, atol=1e-11, h0=0.1, h_max=5.0, lambda_end=800.0,
                                                        n_samples=20))
        assert status[0] == 0
        assert np.abs(s[0, :, 1] - r0).max() <= 1e-6
        assert s[0, -1, 3] / s[0, -1, 0] == pytest.approx(Om, rel=1e-8)
    # the quadrupole changes the orbital frequency in the direction its sign says: oblate (q > 0) mass
    # distributions pull harder in the equatorial plane
    kerr_like = dict(m, q=0.0)
    d = O.kepler_general(m, 7.0, 1.0, 0.0)[0] - O.kepler_general(kerr_like, 7.0, 1.0, 0.0)[0]
    assert d * m["q"] > 0


def test_redshift_factor_side_of_the_disk():
    """g > 1 on the approaching side: for a prograde disk seen with the traced (time-reversed) covector
    that is p_phi > 0 (L_z = -p_phi < 0 ... the photon co-rotates), and g -> the gravitational redshift
    sqrt(-1/g^tt-ish) < 1 for p_phi = 0 far out."""
    for m in (KERR, MN):
        hi = O.kepler_general(m, 8.0, 1.0, +3.0)[2]
        lo = O.kepler_general(m, 8.0, 1.0, -3.0)[2]
        mid = O.kepler_general(m, 8.0, 1.0, 0.0)[2]
        assert lo < mid < hi or hi < mid < lo
        assert 0.6 < mid < 1.0
        assert O.kepler_general(m, 500.0, 1.0, 0.0)[2] == pytest.approx(1.0, abs=5e-3)


def test_disk_trace_with_the_general_emitter():
    """Manko-Novikov image with a thin disk (the paper's Fig 16-17 situation): needs disk_r_in > 0."""
    w = W.workload("C4", width=64, height=64, theta_obs=math.radians(80.0))
    w["cfg"].update(max_steps=3000, max_crossings=3, disk_r_in=4.0, disk_r_out=20.0)
    rec, _ = O.trace(w, 7, None, 5)
    hit = ~np.isnan(rec["disk_r"][:, 0])
    assert 20 < hit.sum() < len(rec)
    assert ((rec["disk_r"][hit, 0] >= 4.0) & (rec["disk_r"][hit, 0] <= 20.0)).all()
    g = rec["disk_g"][hit, 0]
    assert np.isfinite(g).all() and (g > 0.2).all() and (g < 1.8).all() and (g > 1).any() and (g < 1).any()
    w["cfg"]["disk_r_in"] = 0.0
    with pytest.raises(ValueError):
        O.trace(w, 7, 10, 5)
