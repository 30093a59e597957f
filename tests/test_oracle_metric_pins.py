"""Pins for the oracle's point-wise pieces (metric, derivatives, Hamilton's equations, camera,
tableau).  Each test checks the oracle's *own output* against something the mathematics
fixes: vacuum field equations, textbook radii, closed forms, order conditions, brute force.
Citations: P:Lnnn = PAPER.md line; Rn = DESIGN.md section 3 reading.
"""
import math

import numpy as np
import pytest

import gp_workloads as W
from oracle import oracle as O

SCHW = dict(id=0, M=1.0, a=0.0, q=0.0)
KERR = dict(id=1, M=1.0, a=0.9, q=0.0)
MN = dict(id=2, M=1.0, a=0.9, q=0.5)
ALL = [SCHW, KERR, dict(id=1, M=0.7, a=-0.3, q=0.0), MN, dict(id=2, M=1.3, a=0.6, q=-2.0)]
POINTS = [(3.7, 1.1), (10.0, 0.4), (2.5, 2.3), (1000.0, math.pi / 3), (6.0, math.pi / 2)]


def full_matrix(v5):
    gtt, gtp, gpp, grr, gthth = v5
    g = np.zeros((4, 4))  # order t, r, theta, phi
    g[0, 0], g[0, 3], g[3, 0], g[3, 3], g[1, 1], g[2, 2] = gtt, gtp, gtp, gpp, grr, gthth
    return g


# ---- inverse metric is the inverse of the covariant one (eq 3 uses g^{mu nu} of eq 8/9-13/20)
@pytest.mark.parametrize("m", ALL)
def test_inverse_times_covariant_is_identity(m):
    for r, th in POINTS:
        g = full_matrix(O.metric_cov(m, r, th))
        gi = full_matrix(O.metric_inv(m, r, th)[:5])
        assert np.allclose(g @ gi, np.eye(4), atol=1e-10, rtol=0)


# ---- written-out derivatives against brute-force 8th-order central differences of the
# oracle's own inverse metric, and against the complex-step evaluation
def _fd(fun, x, h):
    c = np.array([4 / 5, -1 / 5, 4 / 105, -1 / 280])
    return sum(ck * (fun(x + (k + 1) * h) - fun(x - (k + 1) * h)) for k, ck in enumerate(c)) / h


@pytest.mark.parametrize("m", ALL)
def test_inverse_metric_derivatives(m):
    rh = O.radii(m)[0]
    for r, th in [(1.6 * rh + 0.5, 1.1), (10.0, 0.4), (2.0 * rh + 0.1, 2.3), (30.0, 1.9)]:
        o = O.metric_inv(m, r, th)
        dr = _fd(lambda x: O.metric_inv(m, x, th)[:5], r, 1e-3 * r)
        dth = _fd(lambda x: O.metric_inv(m, r, x)[:5], th, 1e-3)
        scale = np.abs(o[:5]) + 1e-300
        assert np.allclose(o[5:10], dr, rtol=1e-8, atol=1e-9 * scale.max())
        assert np.allclose(o[10:15], dth, rtol=1e-8, atol=1e-9 * scale.max())
        cs = O.metric_inv_complex_step(m, r, th)
        assert np.allclose(o, cs, rtol=1e-11, atol=1e-13 * scale.max())


# ---- Hamilton's equations (eq 102-103, R1): dq = dH/dp, dp = -dH/dq by
# brute-force differences of H = 1/2 g^{mu nu} p_mu p_nu (eq 3) assembled here from the
# oracle's inverse metric
def _H(m, q, p):
    gi = full_matrix(O.metric_inv(m, q[1], q[2])[:5])
    return 0.5 * p @ gi @ p


@pytest.mark.parametrize("m", ALL)
def test_rhs_is_hamiltonian_vector_field(m):
    rng = np.random.default_rng(3)
    rh = O.radii(m)[0]
    for r, th in [(1.6 * rh + 0.5, 1.1), (10.0, 0.4), (2.0 * rh + 0.1, 2.3)]:
        p = rng.normal(size=4)  # p_t, p_r, p_th, p_phi in matrix order t, r, theta, phi
        q = np.array([0.3, r, th, -1.0])
        st = np.array([q[0], q[1], q[2], q[3], p[0], p[1], p[2], p[3]])
        d = O.rhs(m, st)  # dt, dr, dth, dphi, dp_r, dp_th
        for i, want in enumerate([0, 1, 2, 3]):
            e = np.zeros(4)
            e[want] = 1.0
            num = _fd(lambda x: _H(m, q, p + (x - p[want]) * e), p[want], 1e-3)
            assert d[i] == pytest.approx(num, rel=1e-9, abs=1e-11)
        for i, want in ((4, 1), (5, 2)):
            e = np.zeros(4)
            e[want] = 1.0
            num = _fd(lambda x: _H(m, q + (x - q[want]) * e, p), q[want], 1e-3)
            assert d[i] == pytest.approx(-num, rel=1e-8, abs=1e-10)


# ---- Kerr: textbook radii and circular orbits -------------------------------------------
def test_kerr_horizon_isco_values():
    rh, risco = O.radii(KERR)
    assert rh == pytest.approx(1.0 + math.sqrt(1 - 0.81), abs=1e-15)
    # ISCO is the root of r^2 - 6Mr + 8a sqrt(Mr) - 3a^2 (Bardeen, Press & Teukolsky 1972, eq 2.20)
    for a in (0.0, 0.5, 0.9, 0.998):
        m = dict(id=1, M=1.0, a=a, q=0.0) if a else SCHW
        r = O.radii(m)[1]
        assert r * r - 6 * r + 8 * a * math.sqrt(r) - 3 * a * a == pytest.approx(0.0, abs=1e-12)
    assert O.radii(SCHW) == (2.0, pytest.approx(6.0, abs=1e-14))
    assert O.radii(dict(id=1, M=1.0, a=0.998, q=0.0))[1] == pytest.approx(1.2369706551751847, abs=1e-12)
    assert math.isnan(O.radii(MN)[1])
    assert O.radii(MN)[0] == pytest.approx(1.0 + math.sqrt(1 - 0.81), abs=1e-15)  # R24: x = 1


def test_kerr_circular_photon_orbits():
    """r_ph = 2M(1 + cos(2/3 arccos(-+a/M))) (Bardeen 1972): with xi = L/E on Bardeen's critical
    curve and eta = 0 the equatorial orbit has dr = 0 and dp_r = 0."""
    a, M = 0.9, 1.0
    for sign, want in ((-1, 1.557854627), (+1, 3.910267939)):
        r = 2 * M * (1 + math.cos(2 / 3 * math.acos(sign * a / M)))
        assert r == pytest.approx(want, abs=1e-8)
        xi = -(r**3 - 3 * M * r**2 + a * a * r + a * a * M) / (a * (r - M))
        # physical (E, L) = (1, xi) corresponds to the traced covector (p_t, p_phi) = (1, -xi) (R12)
        d = O.rhs(KERR, [0, r, math.pi / 2, 0, 1.0, 0.0, 0.0, -xi])
        assert d[1] == 0.0 and d[2] == 0.0
        assert d[4] == pytest.approx(0.0, abs=1e-12)
        assert d[5] == pytest.approx(0.0, abs=1e-14)
        # null: H = 0
        H = 0.5 * (1.0 * d[0] - xi * d[3])
        assert H == pytest.approx(0.0, abs=1e-12)


def test_schwarzschild_photon_sphere():
    """circular photon orbit at r = 3M with b = L/E = 3 sqrt(3) M; unstable."""
    b = 3 * math.sqrt(3)
    d = O.rhs(SCHW, [0, 3.0, math.pi / 2, 0, 1.0, 0.0, 0.0, b])
    assert d[1] == 0 and d[4] == pytest.approx(0.0, abs=1e-15)
    assert 0.5 * (d[0] + b * d[3]) == pytest.approx(0.0, abs=1e-15)
    assert O.rhs(SCHW, [0, 3.1, math.pi / 2, 0, 1.0, 0.0, 0.0, b])[4] > 0  # pushed outward
    assert O.rhs(SCHW, [0, 2.9, math.pi / 2, 0, 1.0, 0.0, 0.0, b])[4] < 0  # pushed inward


def test_kepler_emitter_against_metric():
    """P:L358-370 (eq 56, R20): a circular equatorial orbit has dp_r = 0; solving that quadratic
    with the oracle's own d_r g^{mu nu} reproduces Omega_K, and u^t follows from g(u,u) = -1
    with the oracle's covariant metric (independent of the closed forms inside orc_kepler)."""
    for m in (dict(id=1, M=1.0, a=0.998, q=0.0), KERR, SCHW, dict(id=1, M=2.0, a=-1.1, q=0.0)):
        for r in (6.0 * m["M"], 9.5 * m["M"], 20.0 * m["M"]):
            Om, ut, g = O.kepler(m, r, 1.0, 0.3)
            o = O.metric_inv(m, r, math.pi / 2)
            # eq 56 with p_t = -1: A l^2 - 2 B l + C = 0 for l = p_phi
            A, B, Cc = o[5 + 2], o[5 + 1], o[5 + 0]
            roots = np.roots([A, -2 * B, Cc])
            cov = O.metric_cov(m, r, math.pi / 2)
            omegas = []
            for l in roots:
                ut_ = o[0] * (-1.0) + o[1] * l
                uphi = o[1] * (-1.0) + o[2] * l
                omegas.append(uphi / ut_)
            assert min(abs(w - Om) for w in omegas) < 1e-12
            ut_norm = 1.0 / math.sqrt(-(cov[0] + 2 * Om * cov[1] + Om * Om * cov[2]))
            assert ut == pytest.approx(ut_norm, rel=1e-12)
            assert g == pytest.approx(1.0 / (ut_norm * (1.0 + Om * 0.3)), rel=1e-12)
    Om, ut, _ = O.kepler(dict(id=1, M=1.0, a=0.998, q=0.0), 6.0, 1.0, 0.0)
    assert Om == pytest.approx(0.06371480861546, abs=1e-13)
    assert ut == pytest.approx(1.33927221892028, abs=1e-12)


def test_schwarzschild_is_kerr_at_zero_spin():
    tiny = dict(id=1, M=1.0, a=1e-13, q=0.0)
    for r, th in POINTS:
        assert np.allclose(O.metric_inv(SCHW, r, th), O.metric_inv(tiny, r, th), rtol=1e-11, atol=1e-12)
        assert np.allclose(O.metric_cov(SCHW, r, th), O.metric_cov(tiny, r, th), rtol=1e-11, atol=1e-12)


# ---- Manko-Novikov --------------------------------------------------------------------------
def test_mn_reduces_to_kerr_at_q0():
    """BASELINE.json: 'q = 0 must reproduce Kerr'.  Fixes R3 (sign of g_tphi) and R4."""
    for a in (0.9, -0.5, 0.3):
        mn0, kerr = dict(id=2, M=1.0, a=a, q=0.0), dict(id=1, M=1.0, a=a, q=0.0)
        for r, th in POINTS:
            assert np.allclose(O.metric_cov(mn0, r, th), O.metric_cov(kerr, r, th), rtol=1e-11, atol=1e-13)
            assert np.allclose(O.metric_inv(mn0, r, th), O.metric_inv(kerr, r, th), rtol=1e-9, atol=1e-12)


def _weyl_fields(m, rho, z):
    """f, omega, gamma of the oracle at Weyl coordinates (rho, z)."""
    M, a = m["M"], m["a"]
    k = math.sqrt(M * M - a * a)
    rp, rm = math.hypot(rho, z + k), math.hypot(rho, z - k)
    x, y = (rp + rm) / (2 * k), (rp - rm) / (2 * k)
    pot = O.mn_potentials(m, M + k * x, math.acos(y))
    return np.array([pot[0], pot[1], 0.5 * math.log(pot[2])])


def _d1(F, x, h):
    c = [4 / 5, -1 / 5, 4 / 105, -1 / 280]
    return sum(ck * (F(x + (k + 1) * h) - F(x - (k + 1) * h)) for k, ck in enumerate(c)) / h


def _d2(F, x, h):
    c = [8 / 5, -1 / 5, 8 / 315, -1 / 560]
    return (-205 / 72 * F(x) + sum(ck * (F(x + (k + 1) * h) + F(x - (k + 1) * h)) for k, ck in enumerate(c))) / (h * h)


@pytest.mark.parametrize("q", [0.0, 0.5, -2.0])
@pytest.mark.parametrize("pt", [(3.1, 1.7), (1.2, -0.8), (0.7, 2.4)])
def test_mn_is_a_vacuum_solution(q, pt):
    """The reading R4-R6 of eq 20-39 must solve Einstein's vacuum equations ('still a
    stationary and axi-symmetric vacuum solution').  In Weyl-Papapetrou form
    ds^2 = -f(dt - w dphi)^2 + f^-1 [e^{2 gamma}(drho^2 + dz^2) + rho^2 dphi^2] these are the Ernst
    equations and two quadratures for gamma; evaluated on the oracle's own f, omega, gamma with
    8th-order differences."""
    m = dict(id=2, M=1.0, a=0.9, q=q)
    rho, z = pt
    h = 0.005  # residual falls as h^8 down to ~1e-9 (rounding) here
    F = lambda r_, z_: _weyl_fields(m, r_, z_)
    v = F(rho, z)
    f, w = v[0], v[1]
    vr, vz = _d1(lambda s: F(s, z), rho, h), _d1(lambda s: F(rho, s), z, h)
    vrr, vzz = _d2(lambda s: F(s, z), rho, h), _d2(lambda s: F(rho, s), z, h)
    lap_f = vrr[0] + vr[0] / rho + vzz[0]
    grad_f2 = vr[0] ** 2 + vz[0] ** 2
    grad_w2 = vr[1] ** 2 + vz[1] ** 2
    # f lap f = |grad f|^2 - f^4 rho^-2 |grad w|^2
    terms = [f * lap_f, grad_f2, f**4 / rho**2 * grad_w2]
    assert terms[0] - terms[1] + terms[2] == pytest.approx(0.0, abs=2e-6 * max(map(abs, terms)) + 1e-10)
    # div(f^2 rho^-2 grad w) = 0  ->  f (w_rr - w_r/rho + w_zz) + 2 (f_r w_r + f_z w_z) = 0
    t2 = [f * (vrr[1] - vr[1] / rho + vzz[1]), 2 * (vr[0] * vr[1] + vz[0] * vz[1])]
    assert t2[0] + t2[1] == pytest.approx(0.0, abs=2e-6 * max(map(abs, t2)) + 1e-10)
    # gamma quadratures
    g_r = rho / (4 * f * f) * (vr[0] ** 2 - vz[0] ** 2) - f * f / (4 * rho) * (vr[1] ** 2 - vz[1] ** 2)
    g_z = rho / (2 * f * f) * vr[0] * vz[0] - f * f / (2 * rho) * vr[1] * vz[1]
    assert vr[2] == pytest.approx(g_r, rel=1e-6, abs=1e-9)
    assert vz[2] == pytest.approx(g_z, rel=1e-6, abs=1e-9)


def test_mn_vacuum_check_detects_a_wrong_sign():
    """The vacuum pin has teeth: Kerr's f with the sign of omega's constant flipped still passes
    (a constant), but scaling omega by 1.01 must fail the first Ernst equation."""
    m = dict(id=2, M=1.0, a=0.9, q=0.5)
    rho, z, h = 1.2, -0.8, 0.02
    F = lambda r_, z_: _weyl_fields(m, r_, z_) * np.array([1.0, 1.01, 1.0])
    v = F(rho, z)
    vr, vz = _d1(lambda s: F(s, z), rho, h), _d1(lambda s: F(rho, s), z, h)
    vrr, vzz = _d2(lambda s: F(s, z), rho, h), _d2(lambda s: F(rho, s), z, h)
    terms = [v[0] * (vrr[0] + vr[0] / rho + vzz[0]), vr[0] ** 2 + vz[0] ** 2,
             v[0] ** 4 / rho**2 * (vr[1] ** 2 + vz[1] ** 2)]
    assert abs(terms[0] - terms[1] + terms[2]) > 1e-4 * max(map(abs, terms))


def test_mn_quadrupole_moment_sign_and_scale():
    """R8: beta = q M^3/k^3 adds a mass quadrupole -q M^3: on the equator
    (f_MN - f_Kerr) r^3 -> -q M^3, on the axis -> +2 q M^3  (q > 0 oblate)."""
    for q in (0.5, -2.0):
        mn, kerr = dict(id=2, M=1.0, a=0.9, q=q), KERR
        for r, tol in ((200.0, 0.02), (800.0, 0.005)):
            de = (-O.metric_cov(mn, r, math.pi / 2)[0] + O.metric_cov(kerr, r, math.pi / 2)[0]) * r**3
            assert de == pytest.approx(-q, rel=tol)
            da = (-O.metric_cov(mn, r, 1e-3)[0] + O.metric_cov(kerr, r, 1e-3)[0]) * r**3
            assert da == pytest.approx(2 * q, rel=tol)


def test_mn_equatorial_reflection_symmetry():
    """'the symmetry of the space in the equator'.  g(r, pi - theta) = g(r, theta) and
    a(x,-y) = -b(x,y) for the potentials of eq 34-35."""
    for r, th in POINTS[:4]:
        assert np.allclose(O.metric_cov(MN, r, th), O.metric_cov(MN, r, math.pi - th), rtol=1e-10)
        p1, p2 = O.mn_potentials(MN, r, th), O.mn_potentials(MN, r, math.pi - th)
        assert p1[6] == pytest.approx(-p2[7], rel=1e-12)


def test_mn_rejects_zero_spin():
    """'we cannot set the spin to exactly 0 ... division by zero' (eq 23)."""
    with pytest.raises(ValueError):
        O.metric_cov(dict(id=2, M=1.0, a=0.0, q=0.5), 5.0, 1.0)


# ---- camera ------------------------------------------------------------------------------
def test_jitter_hash_is_splitmix64():
    """R11: u = (splitmix64_finalise(seed*G + 2*ray + axis) >> 11) * 2^-53.  With a unit window
    of one pixel and amplitude 0.5, alpha = u exactly.  SplitMix64 seeded with 0 outputs
    0xE220A8397B1DCDAF first (Steele, Lea & Flood 2014 reference implementation)."""
    cam = dict(r_obs=10.0, theta_obs=1.0, alpha_min=0.0, alpha_max=1.0, beta_min=0.0, beta_max=1.0,
               width=1, height=1, supersample=1, jitter_seed=0, jitter_amp_px=0.5)
    a, b = O.alpha_beta(cam, [0])[0]
    assert a == (0xE220A8397B1DCDAF >> 11) * 2.0**-53

    def mix(z):
        z = (z + 0x9E3779B97F4A7C15) % 2**64
        z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) % 2**64
        z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) % 2**64
        return z ^ (z >> 31)
    assert b == (mix(1) >> 11) * 2.0**-53
    cam.update(width=7, height=5, alpha_max=7.0, beta_max=5.0, jitter_seed=12345)
    ab = O.alpha_beta(cam, np.arange(35))
    for ray in range(35):
        zx = (12345 * 0x9E3779B97F4A7C15 + 2 * ray) % 2**64
        ux, uy = (mix(zx) >> 11) * 2.0**-53, (mix((zx + 1) % 2**64) >> 11) * 2.0**-53
        assert ab[ray, 0] == (ray % 7 + 0.5) + (2 * ux - 1) * 0.5
        assert ab[ray, 1] == (ray // 7 + 0.5) + (2 * uy - 1) * 0.5


def test_pixel_map_centres_supersample_shift():
    cam = W.workload("C1")["camera"]
    cam.update(jitter_amp_px=0.0, supersample=2)
    ab = O.alpha_beta(cam, [0, 1, 127, 128, 128 * 128 - 1])
    dx = 20.0 / 64
    assert ab[0] == pytest.approx([-10 + 0.25 * dx, -10 + 0.25 * dx], abs=1e-14)
    assert ab[1] == pytest.approx([-10 + 0.75 * dx, -10 + 0.25 * dx], abs=1e-14)
    assert ab[2, 0] == pytest.approx(10 - 0.25 * dx, abs=1e-13)
    assert ab[3] == pytest.approx([-10 + 0.25 * dx, -10 + 0.75 * dx], abs=1e-14)  # J = 0 is beta_min
    assert ab[4] == pytest.approx([10 - 0.25 * dx, 10 - 0.25 * dx], abs=1e-13)
    cam.update(shift_x_px=1e-6, shift_y_px=-2.0)
    ab2 = O.alpha_beta(cam, [0])
    assert ab2[0] == pytest.approx([ab[0, 0] + 1e-6 * dx, ab[0, 1] - 2 * dx], abs=1e-14)


def test_jitter_statistics():
    cam = W.workload("C2")["camera"]
    n = 20000
    ab = O.alpha_beta(cam, np.arange(n))
    cam0 = dict(cam, jitter_amp_px=0.0)
    d = (ab - O.alpha_beta(cam0, np.arange(n))) / (24.0 / 512)
    assert np.all(np.abs(d) <= 0.5)
    assert abs(d.mean()) < 0.01 and d.var() == pytest.approx(1 / 12, rel=0.03)
    assert abs(np.corrcoef(d[:, 0], d[:, 1])[0, 1]) < 0.03


@pytest.mark.parametrize("m", [SCHW, KERR, MN])
def test_initial_covector_is_null_unit_energy_zamo(m):
    """R12 / P:L338-348 (eq 54-55): H = 0; the ZAMO measures energy p.u = 1; the spatial
    direction in the orthonormal frame is the pinhole direction (-r_o, -beta, alpha)/D."""
    cam = dict(W.workload("C2")["camera"], r_obs=40.0, theta_obs=1.0)
    for al, be in ((3.0, -2.0), (-7.5, 0.1), (0.0, 11.0)):
        st = O.initial_state(m, cam, al, be)
        assert st[:4] == pytest.approx([0.0, 40.0, 1.0, 0.0])
        p = np.array([st[4], st[5], st[6], st[7]])
        gi = full_matrix(O.metric_inv(m, 40.0, 1.0)[:5])
        g = O.metric_cov(m, 40.0, 1.0)
        assert 0.5 * p @ gi @ p == pytest.approx(0.0, abs=1e-14)
        Om = -g[1] / g[2]
        zeta = 1 / math.sqrt(-(g[0] + Om * g[1]))
        assert zeta * (p[0] + Om * p[3]) == pytest.approx(1.0, rel=1e-14)
        D = math.sqrt(40.0**2 + al * al + be * be)
        assert p[1] / math.sqrt(g[3]) == pytest.approx(-40.0 / D, rel=1e-14)
        assert p[2] / math.sqrt(g[4]) == pytest.approx(-be / D, rel=1e-14, abs=1e-16)
        assert p[3] / math.sqrt(g[2]) == pytest.approx(al / D, rel=1e-14, abs=1e-16)


def test_image_plane_is_bardeens_at_infinity():
    """R11: alpha = -xi / sin i, beta^2 = eta + a^2 cos^2 i - xi^2 cot^2 i as r_obs -> infinity,
    with xi = L/E = -p_phi/p_t (R12) and eta = Q/E^2."""
    inc = math.radians(60.0)
    cam = dict(W.workload("C2")["camera"], r_obs=1e7, theta_obs=inc)
    for al, be in ((3.0, -2.0), (-7.5, 4.0)):
        st = O.initial_state(KERR, cam, al, be)
        xi = -st[7] / st[4]
        eta = (st[6] ** 2 + math.cos(inc) ** 2 * (st[7] ** 2 / math.sin(inc) ** 2 - 0.81 * st[4] ** 2)) / st[4] ** 2
        assert -xi / math.sin(inc) == pytest.approx(al, rel=1e-6)
        assert eta + 0.81 * math.cos(inc) ** 2 - xi * xi / math.tan(inc) ** 2 == pytest.approx(be * be, rel=1e-5)
        assert (st[6] < 0) == (be > 0)  # beta > 0 looks toward the north pole


# ---- integrator coefficients -------------------------------------------------------------------
def test_dp54_order_conditions():
    """R10: the tableau must be a 5(4) pair: all 17 order conditions up to order 5 for b, the 8
    up to order 4 for b* = b - e (and not the order-5 ones), row sums = c, FSAL row = b."""
    c, a, b, e = O.dp54_tableau()
    assert np.allclose(a.sum(axis=1), c, atol=1e-15)
    assert np.allclose(a[6], b, atol=0) and np.allclose(np.triu(a), 0)
    bs = b - e

    def conds(w):
        ac, ac2, aac = a @ c, a @ c**2, a @ (a @ c)
        return {
            1: [w.sum() - 1],
            2: [w @ c - 1 / 2],
            3: [w @ c**2 - 1 / 3, w @ ac - 1 / 6],
            4: [w @ c**3 - 1 / 4, w @ (c * ac) - 1 / 8, w @ ac2 - 1 / 12, w @ aac - 1 / 24],
            5: [w @ c**4 - 1 / 5, w @ (c**2 * ac) - 1 / 10, w @ (ac * ac) - 1 / 20, w @ (c * ac2) - 1 / 15,
                w @ (a @ c**3) - 1 / 20, w @ (c * aac) - 1 / 30, w @ (a @ (c * ac)) - 1 / 40,
                w @ (a @ ac2) - 1 / 60, w @ (a @ aac) - 1 / 120],
        }
    for order, res in conds(b).items():
        assert np.allclose(res, 0, atol=2e-16 * 8), order
    cs = conds(bs)
    for order in (1, 2, 3, 4):
        assert np.allclose(cs[order], 0, atol=2e-15), order
    assert max(abs(x) for x in cs[5]) > 1e-4


def _reference_flow(m, st, h):
    from scipy.integrate import solve_ivp

    def f(_, y):
        d = O.rhs(m, [y[0], y[1], y[2], y[3], st[4], y[4], y[5], st[7]])
        return d
    y0 = [st[0], st[1], st[2], st[3], st[5], st[6]]
    sol = solve_ivp(f, (0, h), y0, method="DOP853", rtol=1e-13, atol=1e-15)
    return sol.y[:, -1]


@pytest.mark.parametrize("scheme,order", [(0, 4), (2, 5)])
def test_single_step_convergence_order(scheme, order):
    """RK4 (R9) has local error O(h^5); the propagated DP solution O(h^6)."""
    cam = dict(W.workload("C2")["camera"], r_obs=12.0)
    st = O.initial_state(KERR, cam, 4.0, 3.0)
    errs = []
    for h in (0.8, 0.4, 0.2):
        out, _ = O.single_step(KERR, scheme, st, h)
        ref = _reference_flow(KERR, st, h)
        got = np.array([out[0], out[1], out[2], out[3], out[5], out[6]])
        errs.append(np.abs(got - ref).max())
    rates = [math.log2(errs[i] / errs[i + 1]) for i in range(2)]
    assert all(order + 0.5 < r < order + 1.7 for r in rates), (errs, rates)


def test_dp54_error_estimate_scales_as_h5():
    cam = dict(W.workload("C2")["camera"], r_obs=12.0)
    st = O.initial_state(KERR, cam, 4.0, 3.0)
    e = [O.single_step(KERR, 2, st, h)[1] for h in (0.4, 0.2, 0.1)]
    assert 4.5 < math.log2(e[0] / e[1]) < 5.6 and 4.5 < math.log2(e[1] / e[2]) < 5.6
