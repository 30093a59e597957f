"""ctypes binding of the CPU oracle (TEST INFRASTRUCTURE, not the product).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
may import this.  Structures mirror oracle/gp_oracle.h and nothing else.
"""
import ctypes as C
import os

import numpy as np

from . import build as _build

_i64, _f64 = C.c_int64, C.c_double


class OrcMetric(C.Structure):
    _fields_ = [("id", C.c_int32), ("pad_", C.c_int32), ("M", _f64), ("a", _f64), ("q", _f64)]


class OrcCamera(C.Structure):
    _fields_ = [("r_obs", _f64), ("theta_obs", _f64), ("phi_obs", _f64),
                ("alpha_min", _f64), ("alpha_max", _f64), ("beta_min", _f64), ("beta_max", _f64),
                ("width", _i64), ("height", _i64), ("supersample", _i64),
                ("jitter_seed", C.c_uint64),
                ("jitter_amp_px", _f64), ("shift_x_px", _f64), ("shift_y_px", _f64),
                ("projection", _i64), ("focal_2f_over_d", _f64)]


class OrcCfg(C.Structure):
    _fields_ = [("scheme", _i64), ("h", _f64), ("h_rel", _f64), ("rtol", _f64), ("atol", _f64),
                ("h_cap_rel", _f64), ("max_steps", _i64), ("lambda_max", _f64),
                ("eps_capture", _f64), ("r_escape", _f64), ("disk_r_in", _f64),
                ("disk_r_out", _f64), ("max_crossings", _i64), ("ring_half_angle", _f64)]


RECORD_DTYPE = np.dtype([
    ("status", "<i8"), ("n_accepted", "<i8"), ("n_rejected", "<i8"),
    ("n_equator_crossings", "<i8"), ("n_disk_recorded", "<i8"), ("n_rhs", "<i8"),
    ("alpha", "<f8"), ("beta", "<f8"),
    ("t", "<f8"), ("r", "<f8"), ("theta", "<f8"), ("phi", "<f8"),
    ("p_t", "<f8"), ("p_r", "<f8"), ("p_theta", "<f8"), ("p_phi", "<f8"), ("lambda", "<f8"),
    ("h_max", "<f8"), ("q_drift", "<f8"), ("sin_theta_min", "<f8"), ("err_margin", "<f8"),
    ("disk_r", "<f8", (3,)), ("disk_g", "<f8", (3,)),
])
assert RECORD_DTYPE.itemsize == 6 * 8 + 15 * 8 + 6 * 8

_lib = None
_lib_fma = None


def _declare_trace(L):
    L.orc_trace.argtypes = [C.POINTER(OrcMetric), C.POINTER(OrcCamera), C.POINTER(OrcCfg),
                            _i64, _i64, _i64, C.c_void_p, C.c_int]


def lib_rounding_probe():
    """The same oracle source compiled with FMA contraction (oracle/build.py); used only to
    measure the oracle's own rounding sensitivity, never for expected values."""
    global _lib_fma
    if _lib_fma is None:
        _lib_fma = C.CDLL(_build.build_rounding_probe())
        _declare_trace(_lib_fma)
    return _lib_fma


_lib_x87 = None


def lib_rounding_probe_x87():
    """Third rounding sample (x87 build, oracle/build.py); for the threshold study only."""
    global _lib_x87
    if _lib_x87 is None:
        _lib_x87 = C.CDLL(_build.build_rounding_probe_x87())
        _declare_trace(_lib_x87)
    return _lib_x87


def lib():
    global _lib
    if _lib is None:
        path = _build.build()
        L = C.CDLL(path)
        P = C.POINTER
        dp = P(_f64)
        L.orc_alpha_beta.argtypes = [P(OrcCamera), _i64, dp, dp]
        L.orc_alpha_beta.restype = None
        for name in ("orc_metric_cov", "orc_metric_inv", "orc_metric_inv_complex_step",
                     "orc_mn_potentials"):
            f = getattr(L, name)
            f.argtypes = [P(OrcMetric), _f64, _f64, dp]
            f.restype = C.c_int
        L.orc_initial_state.argtypes = [P(OrcMetric), P(OrcCamera), _f64, _f64, dp]
        L.orc_rhs.argtypes = [P(OrcMetric), dp, dp]
        L.orc_radii.argtypes = [P(OrcMetric), dp, dp]
        L.orc_kepler.argtypes = [P(OrcMetric), _f64, _f64, _f64, dp]
        L.orc_dp54_tableau.argtypes = [dp, dp, dp, dp]
        L.orc_dp54_tableau.restype = None
        L.orc_single_step.argtypes = [P(OrcMetric), _i64, dp, _f64, _f64, _f64, dp, dp]
        L.orc_trace.argtypes = [P(OrcMetric), P(OrcCamera), P(OrcCfg), _i64, _i64, _i64,
                                C.c_void_p, C.c_int]
        L.orc_trace_one.argtypes = [P(OrcMetric), P(OrcCamera), P(OrcCfg), _f64, _f64,
                                    C.c_void_p, dp, _i64, P(_i64)]
        _lib = L
    return _lib


def _metric(d):
    return OrcMetric(int(d["id"]), 0, float(d["M"]), float(d.get("a", 0.0)), float(d.get("q", 0.0)))


def _camera(d):
    return OrcCamera(d["r_obs"], d["theta_obs"], d.get("phi_obs", 0.0),
                     d["alpha_min"], d["alpha_max"], d["beta_min"], d["beta_max"],
                     d["width"], d["height"], d.get("supersample", 1), d.get("jitter_seed", 0),
                     d.get("jitter_amp_px", 0.0), d.get("shift_x_px", 0.0), d.get("shift_y_px", 0.0),
                     d.get("projection", 0), d.get("focal_2f_over_d", 0.0))


def _cfg(d):
    return OrcCfg(d["scheme"], d.get("h", 0.0), d.get("h_rel", 0.0), d.get("rtol", 0.0),
                  d.get("atol", 0.0), d.get("h_cap_rel", 0.0), d["max_steps"],
                  d.get("lambda_max", 0.0), d["eps_capture"], d["r_escape"],
                  d.get("disk_r_in", 0.0), d.get("disk_r_out", 0.0), d.get("max_crossings", 0),
                  d.get("ring_half_angle", 0.0))


def _dp(a):
    return a.ctypes.data_as(C.POINTER(_f64))


def _check(rc, what):
    if rc < 0:
        raise ValueError(f"oracle: {what} rejected its arguments (rc={rc})")
    return rc


def alpha_beta(camera, rays):
    cam = _camera(camera)
    rays = np.atleast_1d(np.asarray(rays, dtype=np.int64))
    out = np.empty((rays.size, 2))
    a, b = _f64(), _f64()
    L = lib()
    for i, ray in enumerate(rays):
        L.orc_alpha_beta(C.byref(cam), int(ray), C.byref(a), C.byref(b))
        out[i] = a.value, b.value
    return out


def _point_fn(name, n):
    def fn(metric, r, theta):
        out = np.empty(n)
        _check(getattr(lib(), name)(C.byref(_metric(metric)), float(r), float(theta), _dp(out)), name)
        return out
    fn.__name__ = name
    return fn


metric_cov = _point_fn("orc_metric_cov", 5)
metric_inv = _point_fn("orc_metric_inv", 15)
metric_inv_complex_step = _point_fn("orc_metric_inv_complex_step", 15)
mn_potentials = _point_fn("orc_mn_potentials", 10)


def initial_state(metric, camera, alpha, beta):
    out = np.empty(8)
    _check(lib().orc_initial_state(C.byref(_metric(metric)), C.byref(_camera(camera)),
                                   float(alpha), float(beta), _dp(out)), "initial_state")
    return out


def rhs(metric, state8):
    st = np.ascontiguousarray(state8, dtype=np.float64)
    out = np.empty(6)
    _check(lib().orc_rhs(C.byref(_metric(metric)), _dp(st), _dp(out)), "rhs")
    return out


def radii(metric):
    rh, ri = _f64(), _f64()
    _check(lib().orc_radii(C.byref(_metric(metric)), C.byref(rh), C.byref(ri)), "radii")
    return rh.value, ri.value


def kepler(metric, r, p_t, p_phi):
    out = np.empty(3)
    _check(lib().orc_kepler(C.byref(_metric(metric)), float(r), float(p_t), float(p_phi), _dp(out)), "kepler")
    return out  # Omega_K, u^t, g


def kepler_general(metric, r, p_t, p_phi):
    out = np.empty(3)
    f = lib().orc_kepler_general
    f.argtypes = [C.POINTER(OrcMetric), _f64, _f64, _f64, C.POINTER(_f64)]
    f.restype = C.c_int
    _check(f(C.byref(_metric(metric)), float(r), float(p_t), float(p_phi), _dp(out)), "kepler_general")
    return out  # Omega, u^t, g


def dp54_tableau():
    c, a, b, e = np.empty(7), np.empty(49), np.empty(7), np.empty(7)
    lib().orc_dp54_tableau(_dp(c), _dp(a), _dp(b), _dp(e))
    return c, a.reshape(7, 7), b, e


def single_step(metric, scheme, state8, h, rtol=1e-10, atol=1e-10):
    st = np.ascontiguousarray(state8, dtype=np.float64)
    out, err = np.empty(8), _f64()
    _check(lib().orc_single_step(C.byref(_metric(metric)), int(scheme), _dp(st), float(h),
                                 float(rtol), float(atol), _dp(out), C.byref(err)), "single_step")
    return out, err.value


def trace(workload, ray_begin=0, ray_count=None, ray_stride=1, n_threads=0, rounding_probe=False):
    """Trace rays ray_begin + k*ray_stride of a gp_workloads workload.  Returns
    (records: structured array, threads_used).  rounding_probe=True runs the FMA-contracted
    build of the same source instead (see lib_rounding_probe)."""
    cam = workload["camera"]
    total = cam["width"] * cam["height"] * cam.get("supersample", 1) ** 2
    fit = max(0, (total - ray_begin + ray_stride - 1) // ray_stride)
    if ray_count is None:
        ray_count = fit
    if ray_count > fit:
        raise ValueError("ray selection leaves the image")
    out = np.zeros(ray_count, dtype=RECORD_DTYPE)
    L = (lib_rounding_probe_x87() if rounding_probe == "x87" else lib_rounding_probe()) if rounding_probe else lib()
    used = _check(L.orc_trace(C.byref(_metric(workload["metric"])), C.byref(_camera(cam)),
                                  C.byref(_cfg(workload["cfg"])), int(ray_begin), int(ray_count),
                                  int(ray_stride), out.ctypes.data, int(n_threads)), "trace")
    return out, used


def trace_one(workload, alpha, beta, path_capacity=0):
    """Trace one ray from an explicit image-plane point.  Returns (record, path) where path
    is an (n, 8) array of (lambda, t, r, theta, phi, p_r, p_theta, h) or None."""
    out = np.zeros(1, dtype=RECORD_DTYPE)
    path = np.empty((path_capacity, 8)) if path_capacity else None
    n = _i64(0)
    _check(lib().orc_trace_one(C.byref(_metric(workload["metric"])), C.byref(_camera(workload["camera"])),
                               C.byref(_cfg(workload["cfg"])), float(alpha), float(beta),
                               out.ctypes.data, _dp(path) if path is not None else None,
                               int(path_capacity), C.byref(n)), "trace_one")
    return out[0], (path[: n.value] if path is not None else None)


# ---- image formation (gp_shade_oracle.cpp) --------------------------------------------------------
class OrcShadeCfg(C.Structure):
    _fields_ = [("width", _i64), ("height", _i64), ("supersample", _i64), ("mode", _i64),
                ("grid_step_deg", _f64), ("grid_half_width_deg", _f64),
                ("tex_width", _i64), ("tex_height", _i64), ("tex_seed", C.c_uint64),
                ("time_period", _f64), ("disk_overlay", _i64), ("g_lo", _f64), ("g_hi", _f64)]


def _shade_cfg(d):
    return OrcShadeCfg(d["width"], d["height"], d.get("supersample", 1), d["mode"],
                       d.get("grid_step_deg", 15.0), d.get("grid_half_width_deg", 0.5),
                       d.get("tex_width", 1), d.get("tex_height", 1), d.get("tex_seed", 0),
                       d.get("time_period", 1.0), d.get("disk_overlay", 0), d.get("g_lo", 0.3), d.get("g_hi", 1.5))


def splitmix64(z):
    f = lib().orc_splitmix64
    f.argtypes, f.restype = [C.c_uint64], C.c_uint64
    return f(z)


def canonical_angles(theta, phi):
    out = np.empty(2)
    f = lib().orc_canonical_angles
    f.argtypes, f.restype = [_f64, _f64, C.POINTER(_f64)], None
    f(float(theta), float(phi), _dp(out))
    return out


def shade_ray(cfg, status, theta, phi, t, disk_r0=float("nan"), disk_g0=float("nan")):
    out = np.empty(3)
    f = lib().orc_shade_ray
    f.argtypes, f.restype = [C.POINTER(OrcShadeCfg), _i64, _f64, _f64, _f64, _f64, _f64, C.POINTER(_f64)], None
    f(C.byref(_shade_cfg(cfg)), int(status), float(theta), float(phi), float(t), float(disk_r0), float(disk_g0),
      _dp(out))
    return out


def shade(cfg, status, theta, phi, t, disk_r0=None, disk_g0=None):
    """RGBA8 image (H, W, 4) from per-sub-ray arrays of n = W*H*S*S entries."""
    c = _shade_cfg(cfg)
    n = c.width * c.height * c.supersample ** 2
    st = np.ascontiguousarray(status, dtype=np.int64)
    arr = [np.ascontiguousarray(a, dtype=np.float64) for a in (theta, phi, t)]
    assert st.size == n and all(a.size == n for a in arr)
    dr = np.ascontiguousarray(disk_r0, dtype=np.float64) if disk_r0 is not None else None
    dg = np.ascontiguousarray(disk_g0, dtype=np.float64) if disk_g0 is not None else None
    out = np.zeros((c.height, c.width, 4), dtype=np.uint8)
    f = lib().orc_shade
    P = C.POINTER
    f.argtypes = [P(OrcShadeCfg), P(_i64), P(_f64), P(_f64), P(_f64), P(_f64), P(_f64), C.c_void_p]
    f.restype = C.c_int
    _check(f(C.byref(c), st.ctypes.data_as(P(_i64)), _dp(arr[0]), _dp(arr[1]), _dp(arr[2]),
             _dp(dr) if dr is not None else None, _dp(dg) if dg is not None else None, out.ctypes.data), "shade")
    return out


# ---- orbits from explicit initial states -----------------------------------------------------------
class OrcOrbitCfg(C.Structure):
    _fields_ = [("rtol", _f64), ("atol", _f64), ("h0", _f64), ("h_max", _f64), ("lambda_end", _f64),
                ("eps_capture", _f64), ("n_samples", _i64), ("max_steps", _i64)]


def integrate_orbits(metric, states8, cfg, rounding_probe=False):
    """states8: (n, 8) array (t, r, theta, phi, p_t, p_r, p_theta, p_phi); cfg: dict.  Returns
    (samples (n, n_samples, 8), status (n,), n_steps (n,)).  rounding_probe=True runs the
    FMA-contracted build of the same source (flagging aid only, see lib_rounding_probe)."""
    st = np.ascontiguousarray(states8, dtype=np.float64).reshape(-1, 8)
    n = st.shape[0]
    c = OrcOrbitCfg(cfg["rtol"], cfg["atol"], cfg["h0"], cfg["h_max"], cfg["lambda_end"],
                    cfg.get("eps_capture", 1e-3), cfg["n_samples"], cfg.get("max_steps", 10 ** 7))
    samples = np.empty((n, c.n_samples, 8))
    status = np.zeros(n, dtype=np.int64)
    steps = np.zeros(n, dtype=np.int64)
    f = (lib_rounding_probe() if rounding_probe else lib()).orc_integrate_orbits
    P = C.POINTER
    f.argtypes = [P(OrcMetric), P(OrcOrbitCfg), P(_f64), _i64, P(_f64), P(_i64), P(_i64)]
    f.restype = C.c_int
    _check(f(C.byref(_metric(metric)), C.byref(c), _dp(st), n, _dp(samples), status.ctypes.data_as(P(_i64)),
             steps.ctypes.data_as(P(_i64))), "integrate_orbits")
    return samples, status, steps


def host_threads():
    return os.cpu_count() or 1
