"""ctypes binding of libgp.so — argument marshalling only.

Every entry point has the name and meaning it has in include/gp.h; every step of the method
runs in the CUDA kernels behind it.  There is no CPU path: if the library cannot be loaded the
import of this module raises.  PyTorch appears only as the owner of device memory and streams.
"""
import ctypes as C
import os

import numpy as np

from . import build as _build

HERE = os.path.dirname(os.path.abspath(__file__))

GP_SCHWARZSCHILD, GP_KERR, GP_MANKO_NOVIKOV = 0, 1, 2
GP_RAY_ESCAPED, GP_RAY_CAPTURED, GP_RAY_MAXSTEPS, GP_RAY_NONFINITE, GP_RAY_STEP_UNDERFLOW, GP_RAY_HIT_RING = range(6)
GP_OK, GP_E_BAD_METRIC, GP_E_BAD_PARAM, GP_E_NULL, GP_E_SIZE, GP_E_UNSUPPORTED, GP_E_CUDA, GP_E_STATIC_LIMIT = (
    0, -1, -2, -3, -4, -5, -6, -7)

_f64, _i32, _i64, _u64 = C.c_double, C.c_int32, C.c_int64, C.c_uint64


class gp_metric_params(C.Structure):
    _fields_ = [("M", _f64), ("a", _f64), ("q", _f64)]


class gp_camera(C.Structure):
    _fields_ = [("r_obs", _f64), ("theta_obs", _f64), ("phi_obs", _f64),
                ("alpha_min", _f64), ("alpha_max", _f64), ("beta_min", _f64), ("beta_max", _f64),
                ("width", _i32), ("height", _i32), ("supersample", _i32), ("projection", _i32),
                ("jitter_seed", _u64), ("jitter_amp_px", _f64),
                ("shift_x_px", _f64), ("shift_y_px", _f64),
                ("ray_begin", _i64), ("ray_count", _i64), ("ray_stride", _i64),
                ("focal_2f_over_d", _f64)]


class gp_integrator_cfg(C.Structure):
    _fields_ = [("scheme", _i32), ("precision", _i32),
                ("h", _f64), ("h_rel", _f64), ("rtol", _f64), ("atol", _f64), ("h_cap_rel", _f64),
                ("max_steps", _i64), ("lambda_max", _f64),
                ("eps_capture", _f64), ("r_escape", _f64),
                ("disk_r_in", _f64), ("disk_r_out", _f64),
                ("max_crossings", _i32), ("segment_steps", _i32), ("ring_half_angle", _f64)]


class gp_shade_cfg(C.Structure):
    _fields_ = [("width", _i32), ("height", _i32), ("supersample", _i32), ("mode", _i32),
                ("grid_step_deg", _f64), ("grid_half_width_deg", _f64),
                ("tex_width", _i32), ("tex_height", _i32), ("tex_seed", _u64),
                ("time_period", _f64), ("disk_overlay", _i32), ("reserved_", _i32),
                ("g_lo", _f64), ("g_hi", _f64)]


class gp_orbit_cfg(C.Structure):
    _fields_ = [("rtol", _f64), ("atol", _f64), ("h0", _f64), ("h_max", _f64), ("lambda_end", _f64),
                ("eps_capture", _f64), ("n_samples", _i64), ("max_steps", _i64)]


class gp_out_buffers(C.Structure):
    _fields_ = [("rays", C.c_void_p), ("rays_bytes", C.c_size_t),
                ("disk", C.c_void_p), ("disk_bytes", C.c_size_t),
                ("counters", C.c_void_p), ("counters_bytes", C.c_size_t)]


# numpy views of the record layouts of include/gp.h
RAY_DTYPE = np.dtype([
    ("t", "<f8"), ("r", "<f8"), ("theta", "<f8"), ("phi", "<f8"),
    ("lambda", "<f8"), ("status", "<u4"), ("n_accepted", "<u4"), ("p_r", "<f8"), ("p_theta", "<f8"),
    ("p_t", "<f8"), ("p_phi", "<f8"), ("h_max", "<f8"), ("q_drift", "<f8"),
    ("sin_theta_min", "<f8"), ("err_margin", "<f8"), ("n_rejected", "<u4"),
    ("n_equator_crossings", "<u4"), ("n_disk_recorded", "<u4"), ("n_rhs", "<u4")])
DISK_DTYPE = np.dtype([("r_cross", "<f8", (3,)), ("g", "<f8", (3,))])
assert RAY_DTYPE.itemsize == 128 and DISK_DTYPE.itemsize == 48

EXPORTS = ("gp_integrate_orbits", "gp_shade", "gp_trace", "gp_trace_host", "gp_trace_static", "gp_static_max_rays", "gp_init_conditions", "gp_eval_metric", "gp_eval_rhs",
           "gp_probe_fp64_fma", "gp_metric_radii", "gp_ray_record_size", "gp_disk_record_size",
           "gp_counters_size", "gp_version", "gp_strerror")


def _load():
    path = _build.build()
    if not os.path.exists(path):
        raise ImportError("libgp.so is missing and could not be built: the CUDA library IS the "
                          "product, there is no fallback")
    L = C.CDLL(path)
    P, vp, sz = C.POINTER, C.c_void_p, C.c_size_t
    sig5 = [C.c_int, P(gp_metric_params), P(gp_camera), P(gp_integrator_cfg), P(gp_out_buffers), vp]
    L.gp_trace.argtypes = sig5
    L.gp_trace_host.argtypes = sig5
    L.gp_trace_static.argtypes = sig5
    L.gp_static_max_rays.restype = _i64
    L.gp_static_max_rays.argtypes = []
    L.gp_init_conditions.argtypes = [C.c_int, P(gp_metric_params), P(gp_camera), vp, sz, vp, sz, vp]
    L.gp_eval_metric.argtypes = [C.c_int, P(gp_metric_params), vp, _i64, vp, sz, vp]
    L.gp_eval_rhs.argtypes = [C.c_int, P(gp_metric_params), vp, _i64, vp, sz, vp]
    L.gp_probe_fp64_fma.argtypes = [_i64, vp, sz, P(_f64), vp]
    L.gp_metric_radii.argtypes = [C.c_int, P(gp_metric_params), P(_f64), P(_f64)]
    L.gp_integrate_orbits.argtypes = [C.c_int, P(gp_metric_params), P(gp_orbit_cfg), vp, _i64, vp, sz, vp, sz,
                                      vp, sz, vp]
    L.gp_integrate_orbits.restype = C.c_int
    L.gp_shade.argtypes = [P(gp_shade_cfg), vp, sz, vp, sz, vp, sz, vp]
    L.gp_shade.restype = C.c_int
    for n in ("gp_trace", "gp_trace_host", "gp_trace_static", "gp_init_conditions", "gp_eval_metric", "gp_eval_rhs",
              "gp_probe_fp64_fma", "gp_metric_radii", "gp_version"):
        getattr(L, n).restype = C.c_int
    for n in ("gp_ray_record_size", "gp_disk_record_size", "gp_counters_size"):
        getattr(L, n).restype = sz
        getattr(L, n).argtypes = []
    L.gp_strerror.restype = C.c_char_p
    L.gp_strerror.argtypes = [C.c_int]
    return L


lib = _load()


class GpError(RuntimeError):
    def __init__(self, code, where):
        self.code = code
        super().__init__(f"{where}: {lib.gp_strerror(code).decode()} ({code})")


def _check(code, where):
    if code != GP_OK:
        raise GpError(code, where)


# ---- struct marshalling from the plain dicts of gp_workloads -------------------------------------
def metric_struct(m):
    return gp_metric_params(float(m["M"]), float(m.get("a", 0.0)), float(m.get("q", 0.0)))


def camera_struct(c, ray_begin=0, ray_count=None, ray_stride=1):
    S = int(c.get("supersample", 1))
    total = int(c["width"]) * int(c["height"]) * S * S
    if ray_count is None:
        ray_count = max(0, (total - ray_begin + ray_stride - 1) // ray_stride)
    return gp_camera(c["r_obs"], c["theta_obs"], c.get("phi_obs", 0.0),
                     c["alpha_min"], c["alpha_max"], c["beta_min"], c["beta_max"],
                     int(c["width"]), int(c["height"]), S, int(c.get("projection", 0)),
                     int(c.get("jitter_seed", 0)), c.get("jitter_amp_px", 0.0),
                     c.get("shift_x_px", 0.0), c.get("shift_y_px", 0.0),
                     int(ray_begin), int(ray_count), int(ray_stride), c.get("focal_2f_over_d", 0.0))


def cfg_struct(g):
    return gp_integrator_cfg(int(g["scheme"]), int(g.get("precision", 0)),
                             g.get("h", 0.0), g.get("h_rel", 0.0), g.get("rtol", 0.0),
                             g.get("atol", 0.0), g.get("h_cap_rel", 0.0),
                             int(g["max_steps"]), g.get("lambda_max", 0.0),
                             g["eps_capture"], g["r_escape"],
                             g.get("disk_r_in", 0.0), g.get("disk_r_out", 0.0),
                             int(g.get("max_crossings", 0)), int(g.get("segment_steps", 0)),
                             g.get("ring_half_angle", 0.0))


def _stream_ptr(stream):
    if stream is None:
        import torch
        stream = torch.cuda.current_stream()
    return C.c_void_p(stream.cuda_stream if hasattr(stream, "cuda_stream") else int(stream))


def _dev(t):
    """(pointer, bytes) of a CUDA tensor, (None, 0) for None."""
    if t is None:
        return None, 0
    if not t.is_cuda or not t.is_contiguous():
        raise ValueError("expected a contiguous CUDA tensor")
    return C.c_void_p(t.data_ptr()), t.numel() * t.element_size()


# ---- entry points (same names as include/gp.h) ---------------------------------------------------
def gp_trace(metric_id, metric, camera, cfg, rays, disk, counters, stream=None):
    """Enqueue the trace on `stream`.  metric/camera/cfg: ctypes structs; rays/disk/counters:
    CUDA uint8 tensors owned by the caller (disk may be None)."""
    out = gp_out_buffers()
    out.rays, out.rays_bytes = _dev(rays)
    out.disk, out.disk_bytes = _dev(disk)
    out.counters, out.counters_bytes = _dev(counters)
    _check(lib.gp_trace(int(metric_id), C.byref(metric), C.byref(camera), C.byref(cfg),
                        C.byref(out), _stream_ptr(stream)), "gp_trace")


def gp_trace_host(metric_id, metric, camera, cfg, rays, disk=None, counters=None, stream=None):
    """End-to-end call with HOST numpy buffers (RAY_DTYPE / DISK_DTYPE / 8 x uint64);
    synchronises `stream` before returning."""
    out = gp_out_buffers()
    out.rays, out.rays_bytes = C.c_void_p(rays.ctypes.data), rays.nbytes
    if disk is not None:
        out.disk, out.disk_bytes = C.c_void_p(disk.ctypes.data), disk.nbytes
    if counters is not None:
        out.counters, out.counters_bytes = C.c_void_p(counters.ctypes.data), counters.nbytes
    _check(lib.gp_trace_host(int(metric_id), C.byref(metric), C.byref(camera), C.byref(cfg),
                             C.byref(out), _stream_ptr(stream)), "gp_trace_host")


def gp_trace_static(metric_id, metric, camera, cfg, rays, disk=None, counters=None, stream=None):
    """gp_trace without any allocation: the scratch is the library's static device array (gp.h).
    rays/disk: CUDA uint8 tensors owned by the caller; counters: CUDA tensor of >= 64 bytes or None.
    At most gp_static_max_rays() rays per call; calls that overlap on one GPU race."""
    out = gp_out_buffers()
    out.rays, out.rays_bytes = _dev(rays)
    out.disk, out.disk_bytes = _dev(disk)
    out.counters, out.counters_bytes = _dev(counters)
    _check(lib.gp_trace_static(int(metric_id), C.byref(metric), C.byref(camera), C.byref(cfg),
                               C.byref(out), _stream_ptr(stream)), "gp_trace_static")


def gp_static_max_rays():
    return int(lib.gp_static_max_rays())


def gp_init_conditions(metric_id, metric, camera, states8, alpha_beta2=None, stream=None):
    p, n = _dev(states8)
    q, m = _dev(alpha_beta2)
    _check(lib.gp_init_conditions(int(metric_id), C.byref(metric), C.byref(camera), p, n, q, m,
                                  _stream_ptr(stream)), "gp_init_conditions")


def gp_eval_metric(metric_id, metric, r_theta2, out15, stream=None):
    p, _ = _dev(r_theta2)
    q, m = _dev(out15)
    _check(lib.gp_eval_metric(int(metric_id), C.byref(metric), p, r_theta2.shape[0], q, m,
                              _stream_ptr(stream)), "gp_eval_metric")


def gp_eval_rhs(metric_id, metric, states8, rhs6, stream=None):
    p, _ = _dev(states8)
    q, m = _dev(rhs6)
    _check(lib.gp_eval_rhs(int(metric_id), C.byref(metric), p, states8.shape[0], q, m,
                           _stream_ptr(stream)), "gp_eval_rhs")


def gp_probe_fp64_fma(iters, scratch, stream=None):
    """Enqueue the DFMA-chain probe; returns the flops it issues (time it with events)."""
    p, n = _dev(scratch)
    flops = _f64(0.0)
    _check(lib.gp_probe_fp64_fma(int(iters), p, n, C.byref(flops), _stream_ptr(stream)),
           "gp_probe_fp64_fma")
    return flops.value


def orbit_struct(d):
    return gp_orbit_cfg(d["rtol"], d["atol"], d["h0"], d["h_max"], d["lambda_end"], d.get("eps_capture", 1e-3),
                        int(d["n_samples"]), int(d.get("max_steps", 10 ** 7)))


def gp_integrate_orbits(metric_id, metric, cfg, states8, samples, status, n_steps, stream=None):
    """states8 (n, 8) f64, samples (n, n_samples, 8) f64, status (n,) int32, n_steps (n,) int64: CUDA tensors."""
    p, _ = _dev(states8)
    q, m = _dev(samples)
    r, k = _dev(status)
    u, v = _dev(n_steps)
    _check(lib.gp_integrate_orbits(int(metric_id), C.byref(metric), C.byref(cfg), p, states8.shape[0], q, m, r, k,
                                   u, v, _stream_ptr(stream)), "gp_integrate_orbits")


def shade_struct(d):
    return gp_shade_cfg(int(d["width"]), int(d["height"]), int(d.get("supersample", 1)), int(d["mode"]),
                        d.get("grid_step_deg", 15.0), d.get("grid_half_width_deg", 0.5),
                        int(d.get("tex_width", 1)), int(d.get("tex_height", 1)), int(d.get("tex_seed", 0)),
                        d.get("time_period", 1.0), int(d.get("disk_overlay", 0)), 0,
                        d.get("g_lo", 0.3), d.get("g_hi", 1.5))


def gp_shade(cfg, rays, disk, rgba8, stream=None):
    """Enqueue the image-formation kernel: rays / disk / rgba8 are CUDA uint8 tensors (disk may be None)."""
    p, n = _dev(rays)
    q, m = _dev(disk)
    o, k = _dev(rgba8)
    _check(lib.gp_shade(C.byref(cfg), p, n, q, m, o, k, _stream_ptr(stream)), "gp_shade")


def gp_metric_radii(metric_id, metric):
    rh, ri = _f64(), _f64()
    _check(lib.gp_metric_radii(int(metric_id), C.byref(metric), C.byref(rh), C.byref(ri)),
           "gp_metric_radii")
    return rh.value, ri.value


def gp_ray_record_size():
    return lib.gp_ray_record_size()


def gp_disk_record_size():
    return lib.gp_disk_record_size()


def gp_counters_size():
    return lib.gp_counters_size()


def gp_version():
    return lib.gp_version()


def gp_strerror(code):
    return lib.gp_strerror(int(code)).decode()


# ---- convenience used by tests / bench / smoke: allocate, trace, view ------------------------------
def trace_workload(w, ray_begin=0, ray_count=None, ray_stride=1, stream=None, device="cuda"):
    """Allocate caller-owned device buffers with torch, run gp_trace on a gp_workloads workload
    and return (rays, disk, counters) as numpy structured arrays (after a stream sync)."""
    import torch
    cam = camera_struct(w["camera"], ray_begin, ray_count, ray_stride)
    n = cam.ray_count
    cfg = cfg_struct(w["cfg"])
    rays = torch.empty(max(n, 1) * 128, dtype=torch.uint8, device=device)
    need_disk = cfg.max_crossings > 0 or cfg.ring_half_angle > 0.0
    disk = torch.empty(max(n, 1) * 48, dtype=torch.uint8, device=device) if need_disk else None
    counters = torch.empty(64, dtype=torch.uint8, device=device)
    gp_trace(w["metric"]["id"], metric_struct(w["metric"]), cam, cfg, rays, disk, counters, stream)
    (stream or torch.cuda.current_stream()).synchronize()
    r = rays.cpu().numpy().view(RAY_DTYPE)[:n]
    d = disk.cpu().numpy().view(DISK_DTYPE)[:n] if disk is not None else None
    c = counters.cpu().numpy().view("<u8")
    return r, d, c
