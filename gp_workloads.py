"""Seeded synthetic workloads shared by the CUDA path, the oracle and bench.py.

Plain data only: metric parameters, camera window, integrator settings, ray selection.
This module holds none of the method's arithmetic (the pixel -> (alpha, beta) map with its
SplitMix64 jitter is part of the path, step a2, and is implemented separately on each side).

The paper's workloads are parameter choices plus a pixel grid,
so these configurations *are* the inputs; no dataset or benchmark suite is involved.
C1..C5 follow BASELINE.json `configs[0..4]`; `headline` is configs[1] at 1024x1024, the
configuration BASELINE.json's `metric` is quoted on.
"""
import copy
import math

SCHWARZSCHILD, KERR, MANKO_NOVIKOV = 0, 1, 2


def _camera(r_obs, incl_deg, n, half, jitter=0.5, seed=0, supersample=1):
    return dict(r_obs=float(r_obs), theta_obs=math.radians(incl_deg), phi_obs=0.0,
                alpha_min=-float(half), alpha_max=float(half),
                beta_min=-float(half), beta_max=float(half),
                width=int(n), height=int(n), supersample=int(supersample), projection=0,
                jitter_seed=int(seed), jitter_amp_px=float(jitter),
                shift_x_px=0.0, shift_y_px=0.0)


def _cfg(scheme, h=0.0, h_rel=0.0, rtol=0.0, atol=0.0, h_cap_rel=0.0, max_steps=0,
         r_escape=0.0, eps_capture=1e-3, lambda_max=0.0, disk_r_in=0.0, disk_r_out=0.0,
         max_crossings=0):
    return dict(scheme=int(scheme), precision=0, h=float(h), h_rel=float(h_rel),
                rtol=float(rtol), atol=float(atol), h_cap_rel=float(h_cap_rel),
                max_steps=int(max_steps), lambda_max=float(lambda_max),
                eps_capture=float(eps_capture), r_escape=float(r_escape),
                disk_r_in=float(disk_r_in), disk_r_out=float(disk_r_out),
                max_crossings=int(max_crossings))


_ADAPTIVE = dict(scheme=2, rtol=1e-10, atol=1e-10, h_cap_rel=0.1)

WORKLOADS = {
    # configs[0]: Schwarzschild, fixed-step RK4 h = 0.05, <= 5000 steps
    "C1": dict(metric=dict(id=SCHWARZSCHILD, M=1.0, a=0.0, q=0.0),
               camera=_camera(50.0, 90.0, 64, 10.0),
               cfg=_cfg(0, h=0.05, max_steps=5000, r_escape=100.0)),
    # configs[1]: Kerr a = 0.9, adaptive embedded pair, 512 x 512
    "C2": dict(metric=dict(id=KERR, M=1.0, a=0.9, q=0.0),
               camera=_camera(1000.0, 60.0, 512, 12.0),
               cfg=_cfg(max_steps=1_000_000, r_escape=1100.0, **_ADAPTIVE)),
    # configs[2]: Kerr a = 0.998 with a thin Keplerian disk, 3 recorded crossings
    "C3": dict(metric=dict(id=KERR, M=1.0, a=0.998, q=0.0),
               camera=_camera(1000.0, 80.0, 1024, 25.0, jitter=0.0),
               cfg=_cfg(max_steps=1_000_000, r_escape=1100.0, disk_r_in=0.0, disk_r_out=20.0,
                        max_crossings=3, **_ADAPTIVE)),
    # configs[3]: Manko-Novikov a = 0.9, q = 0.5, equatorial observer, <= 2e5 steps
    "C4": dict(metric=dict(id=MANKO_NOVIKOV, M=1.0, a=0.9, q=0.5),
               camera=_camera(1000.0, 90.0, 2048, 15.0),
               cfg=_cfg(max_steps=200_000, r_escape=1100.0, **_ADAPTIVE)),
    # configs[4]: throughput sweep, RK4 with h = 0.02 r
    "C5a": dict(metric=dict(id=KERR, M=1.0, a=0.9, q=0.0),
                camera=_camera(1000.0, 17.0, 4096, 20.0, jitter=0.0),
                cfg=_cfg(1, h_rel=0.02, max_steps=200_000, r_escape=1100.0)),
    "C5b": dict(metric=dict(id=MANKO_NOVIKOV, M=1.0, a=0.9, q=0.5),
                camera=_camera(1000.0, 60.0, 4096, 20.0, jitter=0.0),
                cfg=_cfg(1, h_rel=0.02, max_steps=200_000, r_escape=1100.0)),
}
# The paper's strongly chaotic case (PAPER.md L418 and Fig 10: Manko-Novikov with Q = 2, S = 0.98 M^2),
# zoomed on the band of long-lived rays at the prograde edge of the shadow: an 8 x 2048 grid of pixel
# centres over alpha in [-2.14, -2.06], beta in [-3.5, 3.5] seen from the equator.  Not one of
# BASELINE.json's configs; it exists so that the chaos flag of configs[3] (companion run shifted by
# 1e-6 px) is raised on some tens of pixels and the statistical comparison runs.
# The step budget is this build's choice (the band's escapers need 1e3-2e4 attempted steps).
WORKLOADS["X3"] = dict(metric=dict(id=MANKO_NOVIKOV, M=1.0, a=0.98, q=2.0),
                       camera=_camera(1000.0, 90.0, 8, 0.0, jitter=0.0),
                       cfg=_cfg(max_steps=20_000, r_escape=1100.0, **_ADAPTIVE))
WORKLOADS["X3"]["camera"].update(width=8, height=2048, alpha_min=-2.14, alpha_max=-2.06,
                                 beta_min=-3.5, beta_max=3.5)
# BASELINE.json `metric`: "1024^2 Kerr a=0.9, FP64" = configs[1] at 1024 x 1024
WORKLOADS["headline"] = copy.deepcopy(WORKLOADS["C2"])
WORKLOADS["headline"]["camera"].update(width=1024, height=1024)
# configs[4]'s fixed-step setup at the headline size, reported beside it
WORKLOADS["headline_rk4"] = copy.deepcopy(WORKLOADS["C5a"])
WORKLOADS["headline_rk4"]["camera"].update(width=1024, height=1024)


def workload(name, **camera_overrides):
    """Deep copy of a named workload; keyword arguments override camera fields."""
    w = copy.deepcopy(WORKLOADS[name])
    w["camera"].update(camera_overrides)
    w["name"] = name
    return w


def n_rays(w):
    c = w["camera"]
    return c["width"] * c["height"] * c["supersample"] ** 2


def ray_selection(w, ray_begin=0, ray_count=None, ray_stride=1):
    """(begin, count, stride) clipped to the image; count None = as many as fit."""
    total = n_rays(w)
    fit = max(0, (total - ray_begin + ray_stride - 1) // ray_stride)
    if ray_count is None or ray_count > fit:
        ray_count = fit
    return int(ray_begin), int(ray_count), int(ray_stride)


def shard(w, rank, world):
    """Multi-GPU partition: cyclic interleave, no exchange step."""
    return ray_selection(w, ray_begin=rank, ray_stride=world)
