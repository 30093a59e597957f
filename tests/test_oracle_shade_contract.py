"""The image-formation oracle against a second, vectorised restatement of the contract text.

`oracle/gp_shade_oracle.cpp` and `csrc/gp_shade.cuh` were written by the same hand from the formulas of
include/gp.h ("image formation"), so a shared misreading of that text would pass the GPU parity test.
This test states the contract a second time, as whole-array numpy expressions written from the header's
sentences (modulo instead of floor-and-subtract for "within a half width of a multiple", the four-weight
form of the bilinear filter, gathers instead of loops), and compares every byte of the oracle's image
on random records: raw angles to +-300 rad, every status code (the ring's 5 included), NaN / finite
first crossings, three modes, S = 1 and 2, with and without the disk overlay.  The two restatements
round differently in the last bit, so a byte may differ by one when 255 x mean + 0.5 falls within 1e-13
of an integer; on 2e5 random values that is not expected to happen and at most one such byte is allowed.
"""
import numpy as np
import pytest

from oracle import oracle as O

PI = np.pi
P8 = np.array([(.85, .25, .25), (.25, .75, .25), (.25, .35, .9), (.9, .8, .2), (.55, .15, .15), (.15, .45, .15),
               (.15, .2, .6), (.6, .5, .1)])
P6 = np.array([(.9, .1, .1), (.9, .6, .1), (.8, .9, .1), (.1, .8, .2), (.1, .5, .9), (.6, .1, .9)])
M64 = np.uint64(0xFFFFFFFFFFFFFFFF)


def splitmix(z):
    z = z.astype(np.uint64)
    with np.errstate(over="ignore"):
        z = z + np.uint64(0x9E3779B97F4A7C15)
        z = (z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
        z = (z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
    return z ^ (z >> np.uint64(31))


def contract(cfg, status, theta, phi, t, r0, g0):
    W, H, S, mode = cfg["width"], cfg["height"], cfg.get("supersample", 1), cfg["mode"]
    n = W * H * S * S
    rgb = np.zeros((n, 3))
    # canonical angles
    th = np.mod(theta, 2 * PI)
    over = th > PI
    th = np.where(over, 2 * PI - th, th)
    ph = np.mod(np.where(over, phi + PI, phi), 2 * PI)
    if mode == 0:
        step, hw = np.deg2rad(cfg["grid_step_deg"]), np.deg2rad(cfg["grid_half_width_deg"])
        quad = np.minimum(3, np.floor(ph / (PI / 2)).astype(int))
        base = P8[4 * (th >= PI / 2) + quad]

        def near(x):
            m = np.mod(x, step)
            return np.minimum(m, step - m) < hw
        rgb[:] = np.where((near(th) | near(ph))[:, None], 0.05, base)
    elif mode == 1:
        tw, thh, seed = cfg["tex_width"], cfg["tex_height"], np.uint64(cfg.get("tex_seed", 0))
        u = ph / (2 * PI) * tw - 0.5
        v = th / PI * thh - 0.5
        i0, j0 = np.floor(u), np.floor(v)
        au, av = (u - i0)[:, None], (v - j0)[:, None]

        def tex(i, j):
            i = np.mod(i.astype(np.int64), tw)
            j = np.clip(j.astype(np.int64), 0, thh - 1)
            with np.errstate(over="ignore"):
                h = splitmix(seed * np.uint64(0x9E3779B97F4A7C15) + (j * tw + i).astype(np.uint64))
            return np.stack([(h >> np.uint64(8 * k)) & np.uint64(0xff) for k in range(3)], 1).astype(float) / 255.0
        rgb[:] = ((1 - au) * (1 - av) * tex(i0, j0) + au * (1 - av) * tex(i0 + 1, j0)
                  + (1 - au) * av * tex(i0, j0 + 1) + au * av * tex(i0 + 1, j0 + 1))
    else:
        rgb[:] = P6[np.floor(np.abs(t) / cfg["time_period"]).astype(np.int64) % 6]
    dark = status != 0
    rgb[dark] = (0.0, 1.0, 1.0) if mode == 2 else (0.0, 0.0, 0.0)
    if cfg.get("disk_overlay", 0):
        have = ~np.isnan(r0)
        lo, hi = cfg.get("g_lo", 0.3), cfg.get("g_hi", 1.5)
        blue, red, white = np.array([0.1, 0.2, 1.0]), np.array([1.0, 0.1, 0.1]), np.ones(3)
        xb = np.clip((g0 - lo) / (1 - lo), 0, 1)[:, None]
        xr = np.clip((g0 - 1) / (hi - 1), 0, 1)[:, None]
        col = np.where((g0 < 1)[:, None], blue + xb * (white - blue), white + xr * (red - white))
        rgb[have] = col[have]
    # box filter over the S x S sub-rays: ray = (j*S + sj)*W*S + (i*S + si)
    mean = rgb.reshape(H, S, W, S, 3).mean(axis=(1, 3))
    out = np.empty((H, W, 4), dtype=np.uint8)
    out[..., :3] = np.clip(np.floor(255 * mean + 0.5), 0, 255).astype(np.uint8)
    out[..., 3] = 255
    return out


@pytest.mark.parametrize("mode", [0, 1, 2])
@pytest.mark.parametrize("S", [1, 2])
@pytest.mark.parametrize("overlay", [0, 1])
def test_oracle_image_equals_the_contract_restated(mode, S, overlay):
    rng = np.random.default_rng(100 * mode + 10 * S + overlay)
    W, H = 96, 64
    n = W * H * S * S
    cfg = dict(width=W, height=H, supersample=S, mode=mode, grid_step_deg=15.0, grid_half_width_deg=0.7,
               tex_width=37, tex_height=19, tex_seed=12345, time_period=13.0, disk_overlay=overlay, g_lo=0.25, g_hi=1.6)
    status = rng.choice([0, 0, 0, 1, 2, 5], n)
    theta = rng.uniform(-300.0, 300.0, n)
    phi = rng.uniform(-300.0, 300.0, n)
    theta[: n // 4] = rng.uniform(0.0, PI, n // 4)           # ordinary exits
    t = rng.uniform(-3000.0, 0.0, n)
    r0 = np.where(rng.random(n) < 0.3, rng.uniform(2.0, 20.0, n), np.nan)
    g0 = np.where(np.isnan(r0), np.nan, rng.uniform(0.05, 2.0, n))
    want = contract(cfg, status, theta, phi, t, r0, g0)
    got = O.shade(cfg, status, theta, phi, t, r0 if overlay else None, g0 if overlay else None)
    diff = np.abs(got.astype(int) - want.astype(int))
    assert diff.max() <= 1 and (diff > 0).sum() <= 1, (int(diff.max()), int((diff > 0).sum()))
    assert (got[..., 3] == 255).all()
    if overlay:
        assert 0.2 < np.isfinite(r0).mean() < 0.4
