"""Image formation through the C-ABI (gp_shade) against oracle/gp_shade_oracle.cpp: byte for byte.

The records shaded come from the ORACLE's trace of the frame (no oracle input ever comes from the CUDA
path): they are packed into the library's 128-byte layout for gp_shade and handed to the shading oracle
as plain arrays.  Synthetic records cover the branches a traced image rarely reaches (raw angles far
outside the principal range, every status, NaN disk slots)."""
import math

import numpy as np
import pytest

import gp_workloads as W

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def gp():
    import paper_2310_15183_b200 as gp
    return gp


@pytest.fixture(scope="module")
def O():
    from oracle import oracle as O
    return O


def records_from_oracle(gp, orc):
    """Oracle trace records -> (gp_ray_record array, gp_disk_record array) in the library's layout."""
    rays = np.zeros(len(orc), dtype=gp.api.RAY_DTYPE)
    for f in ("t", "r", "theta", "phi", "lambda", "p_r", "p_theta", "p_t", "p_phi", "h_max", "q_drift",
              "sin_theta_min", "err_margin"):
        rays[f] = orc[f]
    for f in ("status", "n_accepted", "n_rejected", "n_equator_crossings", "n_disk_recorded", "n_rhs"):
        rays[f] = orc[f].astype(np.uint32)
    disk = np.zeros(len(orc), dtype=gp.api.DISK_DTYPE)
    disk["r_cross"], disk["g"] = orc["disk_r"], orc["disk_g"]
    return rays, disk


def gpu_shade(gp, cfg, rays_np, disk_np=None):
    import torch
    rays = torch.from_numpy(rays_np.view(np.uint8).copy()).cuda()
    disk = torch.from_numpy(disk_np.view(np.uint8).copy()).cuda() if disk_np is not None else None
    out = torch.zeros(cfg["height"] * cfg["width"] * 4, dtype=torch.uint8, device="cuda")
    gp.gp_shade(gp.api.shade_struct(cfg), rays, disk, out)
    torch.cuda.synchronize()
    return out.cpu().numpy().reshape(cfg["height"], cfg["width"], 4)


def oracle_shade(O, cfg, rays_np, disk_np=None):
    return O.shade(cfg, rays_np["status"].astype(np.int64), rays_np["theta"], rays_np["phi"], rays_np["t"],
                   disk_np["r_cross"][:, 0] if disk_np is not None else None,
                   disk_np["g"][:, 0] if disk_np is not None else None)


MODES = [dict(mode=0, grid_step_deg=15.0, grid_half_width_deg=0.4),
         dict(mode=1, tex_width=256, tex_height=128, tex_seed=3),
         dict(mode=2, time_period=3.0)]


@pytest.mark.parametrize("mode", MODES, ids=["grid", "texture", "bands"])
@pytest.mark.parametrize("S", [1, 2])
def test_shade_traced_kerr_image_is_bit_exact(gp, O, mode, S):
    w = W.workload("C2", width=192, height=160, supersample=S)
    rays, _ = records_from_oracle(gp, O.trace(w)[0])
    cfg = dict(width=192, height=160, supersample=S, **mode)
    img = gpu_shade(gp, cfg, rays)
    ref = oracle_shade(O, cfg, rays)
    assert img.shape == ref.shape == (160, 192, 4)
    assert np.array_equal(img, ref), f"{np.count_nonzero((img != ref).any(axis=2))} pixels differ"
    assert (img[..., 3] == 255).all()
    shadow = rays["status"].reshape(160 * S, 192 * S)[::S, ::S] != 0
    assert 0.02 < shadow.mean() < 0.5           # the image does contain a shadow and a sky
    assert len(np.unique(img.reshape(-1, 4), axis=0)) > (3 if mode["mode"] != 1 else 100)


def test_shade_disk_overlay_is_bit_exact(gp, O):
    w = W.workload("C3", width=256, height=256)
    rays, disk = records_from_oracle(gp, O.trace(w)[0])
    cfg = dict(width=256, height=256, mode=0, grid_step_deg=10.0, grid_half_width_deg=0.3, disk_overlay=1,
               g_lo=0.2, g_hi=1.6)
    img = gpu_shade(gp, cfg, rays, disk)
    ref = oracle_shade(O, cfg, rays, disk)
    assert np.array_equal(img, ref)
    hit = ~np.isnan(disk["r_cross"][:, 0])
    assert 0.001 < hit.mean() < 0.5
    # the approaching side of the disk is blue-shifted... here g > 1 is drawn red
    g = disk["g"][hit, 0]
    assert (g > 1).any() and (g < 1).any()


def test_shade_synthetic_records_cover_every_branch(gp, O):
    rng = np.random.default_rng(5)
    Wd, Hd, S = 96, 64, 2
    n = Wd * Hd * S * S
    rays = np.zeros(n, dtype=gp.api.RAY_DTYPE)
    rays["status"] = rng.choice([0, 0, 0, 0, 1, 2, 3, 4], n)
    rays["theta"] = rng.uniform(-15.0, 15.0, n)          # raw, accumulated angles
    rays["phi"] = rng.uniform(-300.0, 300.0, n)
    rays["t"] = -rng.uniform(0.0, 5000.0, n)
    # exact boundary values: poles, seam, quadrant edges, multiples of the grid step
    edge = rng.choice(n, 400, replace=False)
    rays["theta"][edge] = rng.choice([0.0, math.pi, math.pi / 2, -math.pi, 2 * math.pi, math.pi / 12 * 5], 400)
    rays["phi"][edge] = rng.choice([0.0, math.pi / 2, math.pi, 2 * math.pi, -math.pi / 2, math.pi / 12 * 7], 400)
    disk = np.zeros(n, dtype=gp.api.DISK_DTYPE)
    disk["r_cross"][:] = np.nan
    disk["g"][:] = np.nan
    hit = rng.random(n) < 0.3
    disk["r_cross"][hit, 0] = rng.uniform(1.3, 20.0, hit.sum())
    disk["g"][hit, 0] = rng.uniform(0.05, 2.0, hit.sum())
    for mode in MODES:
        for overlay in (0, 1):
            cfg = dict(width=Wd, height=Hd, supersample=S, disk_overlay=overlay, g_lo=0.3, g_hi=1.5, **mode)
            img = gpu_shade(gp, cfg, rays, disk if overlay else None)
            ref = oracle_shade(O, cfg, rays, disk if overlay else None)
            assert np.array_equal(img, ref), (mode, overlay, np.count_nonzero((img != ref).any(axis=2)))


def test_shade_validation(gp):
    import torch
    rays = torch.zeros(16 * 128, dtype=torch.uint8, device="cuda")
    out = torch.zeros(16 * 4, dtype=torch.uint8, device="cuda")
    ok = dict(width=4, height=4, mode=0)
    gp.gp_shade(gp.api.shade_struct(ok), rays, None, out)
    for bad, code in ((dict(ok, mode=3), gp.api.GP_E_BAD_PARAM), (dict(ok, width=0), gp.api.GP_E_BAD_PARAM),
                      (dict(ok, grid_step_deg=0.0), gp.api.GP_E_BAD_PARAM),
                      (dict(ok, mode=2, time_period=0.0), gp.api.GP_E_BAD_PARAM),
                      (dict(ok, mode=1, tex_width=0), gp.api.GP_E_BAD_PARAM),
                      (dict(ok, width=8), gp.api.GP_E_SIZE), (dict(ok, disk_overlay=1), gp.api.GP_E_NULL)):
        with pytest.raises(gp.api.GpError) as e:
            gp.gp_shade(gp.api.shade_struct(bad), rays, None, out)
        assert e.value.code == code, bad
    torch.cuda.synchronize()
