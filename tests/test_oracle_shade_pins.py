"""Pins of the image-formation oracle (oracle/gp_shade_oracle.cpp) against what the formulas of
include/gp.h ("image formation") and plain mathematics fix.  CPU only."""
import math

import numpy as np
import pytest

from oracle import oracle as O

PAL8 = [(.85, .25, .25), (.25, .75, .25), (.25, .35, .9), (.9, .8, .2),
        (.55, .15, .15), (.15, .45, .15), (.15, .2, .6), (.6, .5, .1)]
PAL6 = [(.9, .1, .1), (.9, .6, .1), (.8, .9, .1), (.1, .8, .2), (.1, .5, .9), (.6, .1, .9)]
GRID = dict(width=1, height=1, mode=0, grid_step_deg=15.0, grid_half_width_deg=0.5)


def test_splitmix64_reference_vector():
    # first outputs of the SplitMix64 generator seeded with 0 (Steele, Lea & Flood 2014; the values
    # printed by the public-domain reference implementation): the state advances by the golden gamma
    # and orc_splitmix64(z) adds it itself, so output k is orc_splitmix64(k * gamma).
    gamma = 0x9E3779B97F4A7C15
    want = [0xE220A8397B1DCDAF, 0x6E789E6AA1B965F4, 0x06C45D188009454F]
    got = [O.splitmix64((k * gamma) % 2 ** 64) for k in range(3)]
    assert got == want


@pytest.mark.parametrize("theta,phi", [(0.3, 1.0), (-0.3, 1.0), (3.5, -2.0), (7.0, 40.0), (-9.1, -0.2),
                                       (2 * math.pi + 1.2, 5.0)])
def test_canonical_angles_point_at_the_same_direction(theta, phi):
    th, ph = O.canonical_angles(theta, phi)
    assert 0.0 <= th <= math.pi and 0.0 <= ph < 2 * math.pi
    raw = (math.sin(theta) * math.cos(phi), math.sin(theta) * math.sin(phi), math.cos(theta))
    can = (math.sin(th) * math.cos(ph), math.sin(th) * math.sin(ph), math.cos(th))
    assert np.allclose(raw, can, atol=1e-14)
    # and against the transcendental route acos(cos theta), atan2
    assert th == pytest.approx(math.acos(math.cos(theta)), abs=1e-14)
    want_ph = math.atan2(raw[1], raw[0]) % (2 * math.pi)
    assert min(abs(ph - want_ph), 2 * math.pi - abs(ph - want_ph)) <= 1e-13


def test_celestial_grid_palette_and_lines():
    deg = math.pi / 180
    # one point in every octant, well away from the 15-degree lines
    for hemi, th in ((0, 50 * deg), (1, 130 * deg)):
        for q in range(4):
            ph = (q * 90 + 40) * deg
            assert tuple(O.shade_ray(GRID, 0, th, ph, 0.0)) == PAL8[4 * hemi + q]
    # on a meridian (phi = 45 deg) and on a parallel (theta = 60 deg): the line colour
    assert tuple(O.shade_ray(GRID, 0, 50 * deg, 45.2 * deg, 0.0)) == (.05, .05, .05)
    assert tuple(O.shade_ray(GRID, 0, 59.7 * deg, 40 * deg, 0.0)) == (.05, .05, .05)
    assert tuple(O.shade_ray(GRID, 0, 59.4 * deg, 40 * deg, 0.0)) == PAL8[0]   # 0.6 deg off: not a line
    # shadow: black in modes 0 and 1, cyan in the exit-time map
    for status in (1, 2, 3, 4):
        assert tuple(O.shade_ray(GRID, status, 1.0, 1.0, 0.0)) == (0.0, 0.0, 0.0)
        assert tuple(O.shade_ray(dict(GRID, mode=2, time_period=5.0), status, 1.0, 1.0, 0.0)) == (0.0, 1.0, 1.0)


def test_exit_time_bands():
    cfg = dict(width=1, height=1, mode=2, time_period=7.5)
    for t, band in ((0.0, 0), (-7.4, 0), (-7.6, 1), (-2107.3, int(2107.3 // 7.5)), (44.9, 5), (45.1, 6)):
        assert tuple(O.shade_ray(cfg, 0, 1.0, 1.0, t)) == PAL6[band % 6]


def _texel(seed, tw, i, j):
    h = O.splitmix64((seed * 0x9E3779B97F4A7C15 + j * tw + i) % 2 ** 64)
    return np.array([h & 0xff, (h >> 8) & 0xff, (h >> 16) & 0xff]) / 255.0


def test_texture_bilinear_filter():
    cfg = dict(width=1, height=1, mode=1, tex_width=64, tex_height=32, tex_seed=7)
    tw, th_ = 64, 32
    # at a texel centre the sample is the texel
    for i, j in ((0, 0), (5, 9), (63, 31), (31, 16)):
        ph, th = (i + 0.5) / tw * 2 * math.pi, (j + 0.5) / th_ * math.pi
        assert np.allclose(O.shade_ray(cfg, 0, th, ph, 0.0), _texel(7, tw, i, j), atol=1e-14)
    # half-way between four texels: their mean; across the phi seam the column wraps
    ph, th = 6.0 / tw * 2 * math.pi, 10.0 / th_ * math.pi
    mean = sum(_texel(7, tw, i, j) for i in (5, 6) for j in (9, 10)) / 4
    assert np.allclose(O.shade_ray(cfg, 0, th, ph, 0.0), mean, atol=1e-13)
    ph = 1e-9
    seam = (_texel(7, tw, 63, 9) + _texel(7, tw, 0, 9) + _texel(7, tw, 63, 10) + _texel(7, tw, 0, 10)) / 4
    assert np.allclose(O.shade_ray(cfg, 0, th, ph, 0.0), seam, atol=1e-9)
    # near the pole the row index clamps: independent of theta above the first texel centre
    a = O.shade_ray(cfg, 0, 0.1 / th_ * math.pi, 1.0, 0.0)
    b = O.shade_ray(cfg, 0, 0.4 / th_ * math.pi, 1.0, 0.0)
    assert np.allclose(a, b, atol=1e-14)
    # random points against a numpy gather of the same definition
    rng = np.random.default_rng(0)
    for _ in range(200):
        th, ph = rng.uniform(0, math.pi), rng.uniform(0, 2 * math.pi)
        u, v = ph / (2 * math.pi) * tw - 0.5, th / math.pi * th_ - 0.5
        i0, j0 = math.floor(u), math.floor(v)
        au, av = u - i0, v - j0
        cl = lambda j: min(max(j, 0), th_ - 1)
        top = (1 - au) * _texel(7, tw, i0 % tw, cl(j0)) + au * _texel(7, tw, (i0 + 1) % tw, cl(j0))
        bot = (1 - au) * _texel(7, tw, i0 % tw, cl(j0 + 1)) + au * _texel(7, tw, (i0 + 1) % tw, cl(j0 + 1))
        assert np.allclose(O.shade_ray(cfg, 0, th, ph, 0.0), (1 - av) * top + av * bot, atol=1e-13)


def test_disk_colour_map_and_precedence():
    cfg = dict(GRID, disk_overlay=1, g_lo=0.3, g_hi=1.5)
    assert np.allclose(O.shade_ray(cfg, 0, 1.0, 1.0, 0.0, 6.0, 1.0), (1, 1, 1))
    assert np.allclose(O.shade_ray(cfg, 0, 1.0, 1.0, 0.0, 6.0, 0.3), (.1, .2, 1))
    assert np.allclose(O.shade_ray(cfg, 0, 1.0, 1.0, 0.0, 6.0, 0.1), (.1, .2, 1))          # clamped
    assert np.allclose(O.shade_ray(cfg, 0, 1.0, 1.0, 0.0, 6.0, 1.5), (1, .1, .1))
    assert np.allclose(O.shade_ray(cfg, 0, 1.0, 1.0, 0.0, 6.0, 1.25), (1, .55, .55))
    assert np.allclose(O.shade_ray(cfg, 0, 1.0, 1.0, 0.0, 6.0, 0.65), (.55, .6, 1))
    # the disk is opaque: a captured ray that crossed it shows the disk; no crossing -> background
    assert np.allclose(O.shade_ray(cfg, 1, 1.0, 1.0, 0.0, 6.0, 1.0), (1, 1, 1))
    assert tuple(O.shade_ray(cfg, 1, 1.0, 1.0, 0.0)) == (0.0, 0.0, 0.0)
    assert tuple(O.shade_ray(dict(cfg, disk_overlay=0), 0, 50 * math.pi / 180, 40 * math.pi / 180, 0.0, 6.0, 1.0)) == PAL8[0]


def test_image_assembly_quantisation_and_supersampling():
    deg = math.pi / 180
    # 2 x 1 image, S = 2: pixel 0 all captured, pixel 1 half octant 0 and half captured
    cfg = dict(GRID, width=2, height=1, supersample=2)
    status = np.array([1, 1, 0, 1,
                       1, 1, 0, 1])          # rows of the 4 x 2 supersampled grid
    theta = np.full(8, 50 * deg)
    phi = np.full(8, 40 * deg)
    img = O.shade(cfg, status, theta, phi, np.zeros(8))
    assert img.shape == (1, 2, 4)
    assert tuple(img[0, 0]) == (0, 0, 0, 255)
    want = [math.floor(255 * (2 * c / 4) + 0.5) for c in PAL8[0]]
    assert tuple(img[0, 1]) == (*want, 255)
    # identical sub-rays: supersampling changes nothing
    one = O.shade(dict(GRID, width=1, height=1), [0], [50 * deg], [40 * deg], [0.0])
    four = O.shade(dict(GRID, width=1, height=1, supersample=2), [0] * 4, [50 * deg] * 4, [40 * deg] * 4, [0.0] * 4)
    assert np.array_equal(one, four)
    assert tuple(one[0, 0]) == (217, 64, 64, 255)      # floor(255 * (.85, .25, .25) + .5)
