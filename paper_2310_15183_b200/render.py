"""Render a frame: trace every pixel's geodesic, colour the exit states, write an image file.

    python -m paper_2310_15183_b200.render --workload C3 --size 512 --mode grid --disk --out kerr_disk.png

The two steps of the paper's program (the data-generating script and the drawing
script) through this library's C-ABI: gp_trace into device records, gp_shade into an RGBA8 device
buffer, one device-to-host copy of the pixels.  No graphics API: the image is a headless buffer written
as PNG (zlib from the standard library) or binary PPM.  Argument marshalling only — every step runs in
the CUDA kernels.
"""
import argparse
import math
import struct
import sys
import zlib


def write_png(path, rgba):
    """rgba: (H, W, 4) uint8 numpy array."""
    h, w, _ = rgba.shape
    raw = b"".join(b"\x00" + rgba[j].tobytes() for j in range(h))

    def chunk(tag, data):
        return struct.pack(">I", len(data)) + tag + data + struct.pack(">I", zlib.crc32(tag + data) & 0xffffffff)
    with open(path, "wb") as f:
        f.write(b"\x89PNG\r\n\x1a\n" + chunk(b"IHDR", struct.pack(">IIBBBBB", w, h, 8, 6, 0, 0, 0)) +
                chunk(b"IDAT", zlib.compress(raw, 6)) + chunk(b"IEND", b""))


def write_ppm(path, rgba):
    h, w, _ = rgba.shape
    with open(path, "wb") as f:
        f.write(b"P6\n%d %d\n255\n" % (w, h) + rgba[..., :3].tobytes())


def render(workload, size=None, supersample=1, mode="grid", disk=False, inclination_deg=None, projection=0,
           tex=(2048, 1024), time_period=25.0, device="cuda", ring_half_angle=0.0):
    """Returns ((H, W, 4) uint8 image with row 0 at the top, dict of timings and counters)."""
    import numpy as np
    import torch
    import gp_workloads as W
    from . import api

    over = {}
    if size:
        over.update(width=size, height=size)
    if inclination_deg is not None:
        over.update(theta_obs=math.radians(inclination_deg))
    w = W.workload(workload, supersample=supersample, projection=projection, **over)
    cfg = api.cfg_struct(w["cfg"])
    if disk and cfg.max_crossings == 0:
        w["cfg"].update(max_crossings=1, disk_r_out=20.0,
                        disk_r_in=(4.0 if w["metric"]["id"] == W.MANKO_NOVIKOV else 0.0))
        cfg = api.cfg_struct(w["cfg"])
    if ring_half_angle > 0.0:      # the paper's solid ring (Figs 15-17) instead of the thin disk
        w["cfg"].update(max_crossings=0, ring_half_angle=ring_half_angle, disk_r_out=14.0,
                        disk_r_in=(5.0 if w["metric"]["id"] == W.MANKO_NOVIKOV else 0.0))
        cfg = api.cfg_struct(w["cfg"])
    cam = api.camera_struct(w["camera"])
    n = cam.ray_count
    W_, H_ = w["camera"]["width"], w["camera"]["height"]
    rays = torch.empty(n * 128, dtype=torch.uint8, device=device)
    need_disk = cfg.max_crossings > 0 or cfg.ring_half_angle > 0.0
    drec = torch.empty(n * 48, dtype=torch.uint8, device=device) if need_disk else None
    counters = torch.empty(64, dtype=torch.uint8, device=device)
    out = torch.empty(W_ * H_ * 4, dtype=torch.uint8, device=device)
    stream = torch.cuda.current_stream()
    e = [torch.cuda.Event(enable_timing=True) for _ in range(3)]
    e[0].record(stream)
    api.gp_trace(w["metric"]["id"], api.metric_struct(w["metric"]), cam, cfg, rays, drec, counters, stream)
    e[1].record(stream)
    scfg = api.shade_struct(dict(width=W_, height=H_, supersample=supersample,
                                 mode={"grid": 0, "texture": 1, "time": 2}[mode], grid_step_deg=15.0,
                                 grid_half_width_deg=0.6, tex_width=tex[0], tex_height=tex[1], tex_seed=1,
                                 time_period=time_period, disk_overlay=int(drec is not None), g_lo=0.3, g_hi=1.6))
    api.gp_shade(scfg, rays, drec, out, stream)
    e[2].record(stream)
    stream.synchronize()
    img = out.cpu().numpy().reshape(H_, W_, 4)[::-1]      # row j = 0 is beta_min: flip so that north is up
    cnt = counters.cpu().numpy().view("<u8")
    info = dict(rays=int(n), trace_ms=e[0].elapsed_time(e[1]), shade_ms=e[1].elapsed_time(e[2]),
                attempted_steps=int(cnt[2]), rhs_evaluations=int(cnt[3]))
    return np.ascontiguousarray(img), info


def main(argv=None):
    ap = argparse.ArgumentParser(description=__doc__, formatter_class=argparse.RawDescriptionHelpFormatter)
    ap.add_argument("--workload", default="C2", help="a gp_workloads name: C1..C5b, headline, headline_rk4")
    ap.add_argument("--size", type=int, default=512, help="image is size x size pixels")
    ap.add_argument("--supersample", type=int, default=1)
    ap.add_argument("--mode", default="grid", choices=["grid", "texture", "time"])
    ap.add_argument("--disk", action="store_true", help="thin Keplerian disk coloured by its redshift factor")
    ap.add_argument("--ring", type=float, default=0.0, metavar="HALF_ANGLE",
                    help="solid ring of that half opening angle (rad) about the equator, coloured by redshift (adaptive workloads)")
    ap.add_argument("--inclination", type=float, default=None, help="observer polar angle in degrees")
    ap.add_argument("--screen-camera", action="store_true", help="the paper's Euclidean-screen camera (parallel rays)")
    ap.add_argument("--out", default="frame.png", help=".png or .ppm")
    a = ap.parse_args(argv)
    img, info = render(a.workload, a.size, a.supersample, a.mode, a.disk, a.inclination, int(a.screen_camera),
                       ring_half_angle=a.ring)
    (write_ppm if a.out.lower().endswith(".ppm") else write_png)(a.out, img)
    print(f"{a.out}: {img.shape[1]}x{img.shape[0]}, {info['rays']} rays, trace {info['trace_ms']:.2f} ms, "
          f"shade {info['shade_ms']:.3f} ms, {info['rhs_evaluations']} RHS evaluations", file=sys.stderr)
    return 0


if __name__ == "__main__":
    raise SystemExit(main())
