"""CPU-side checks of the C-ABI boundary: libgp.so builds for sm_100a, loads, exports every
symbol include/gp.h declares, keeps the documented record layouts, validates arguments
synchronously, and FAILS LOUDLY (GP_E_CUDA) instead of falling back when no GPU is present.
No kernel is launched here.
"""
import ctypes as C
import math
import os
import re
import subprocess

import numpy as np
import pytest

import gp_workloads as W
import paper_2310_15183_b200 as gp
from paper_2310_15183_b200 import api

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "gp.h")


def _declared_functions():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(gp_[a-z0-9_]+)\s*\(", src)))


def test_every_declared_symbol_is_exported():
    names = _declared_functions()
    assert "gp_trace" in names and "gp_trace_host" in names and len(names) >= 12
    lib = C.CDLL(os.path.join(ROOT, "paper_2310_15183_b200", "libgp.so"))
    for n in names:
        assert hasattr(lib, n), f"{n} declared in gp.h but not exported by libgp.so"
    assert set(names) == set(api.EXPORTS)
    for n in names:
        assert callable(getattr(gp, n)), f"binding lacks {n}"


def test_library_is_sm100a_native_cuda():
    """The binary carries sm_100a SASS for both integrator kernels (no PTX-only JIT path)."""
    out = subprocess.run(["cuobjdump", "-lelf", os.path.join(ROOT, "paper_2310_15183_b200", "libgp.so")],
                         capture_output=True, text=True)
    if out.returncode != 0:
        pytest.skip("cuobjdump unavailable")
    assert "sm_100a" in out.stdout


def test_record_layouts():
    assert gp.gp_ray_record_size() == 128 == api.RAY_DTYPE.itemsize
    assert gp.gp_disk_record_size() == 48 == api.DISK_DTYPE.itemsize
    assert gp.gp_counters_size() == 64
    assert gp.gp_version() == 103
    f = api.RAY_DTYPE.fields
    assert f["lambda"][1] == 32 and f["status"][1] == 40 and f["p_r"][1] == 48 and f["p_t"][1] == 64
    assert f["sin_theta_min"][1] == 96 and f["err_margin"][1] == 104 and f["n_rhs"][1] == 124
    assert C.sizeof(api.gp_camera) == 7 * 8 + 4 * 4 + 8 + 3 * 8 + 3 * 8 + 8
    assert C.sizeof(api.gp_integrator_cfg) == 8 + 5 * 8 + 8 + 8 + 2 * 8 + 2 * 8 + 8 + 8


def test_strerror():
    assert gp.gp_strerror(0) == "ok"
    for code in range(-7, 0):
        assert gp.gp_strerror(code) not in ("ok", "unknown error code")
    assert "GP_STATIC_MAX_RAYS (1048576)" in gp.gp_strerror(api.GP_E_STATIC_LIMIT)
    assert gp.gp_strerror(-99) == "unknown error code"


def test_metric_radii_closed_forms():
    """r_+ = M + sqrt(M^2 - a^2) and the Bardeen-Press-Teukolsky prograde ISCO (values computed
    independently with mpmath during the survey, SURVEY.md pin P11)."""
    rh, ri = gp.gp_metric_radii(gp.GP_KERR, api.gp_metric_params(1.0, 0.9, 0.0))
    assert rh == pytest.approx(1.435889894354067, abs=1e-15)
    assert ri == pytest.approx(2.320883041761887, abs=1e-14)
    rh, ri = gp.gp_metric_radii(gp.GP_KERR, api.gp_metric_params(1.0, 0.998, 0.0))
    assert rh == pytest.approx(1.063213922517116, abs=1e-15)
    assert ri == pytest.approx(1.236970655175184, abs=1e-13)
    rh, ri = gp.gp_metric_radii(gp.GP_SCHWARZSCHILD, api.gp_metric_params(1.0, 0.3, 0.0))
    assert rh == 2.0 and ri == pytest.approx(6.0, abs=1e-14)
    rh, ri = gp.gp_metric_radii(gp.GP_MANKO_NOVIKOV, api.gp_metric_params(1.0, 0.9, 0.5))
    assert rh == pytest.approx(1.4358898943540674, abs=1e-15) and math.isnan(ri)


def _call(w, mutate=None, metric_id=None, out=None, entry="gp_trace"):
    m = api.metric_struct(w["metric"])
    cam = api.camera_struct(w["camera"], 0, 64, 1)
    cfg = api.cfg_struct(w["cfg"])
    if mutate:
        mutate(m, cam, cfg)
    if out is None:
        out = api.gp_out_buffers(C.c_void_p(0x1000), 64 * 128, C.c_void_p(0x2000), 64 * 48,
                                 C.c_void_p(0x3000), 64)
    mid = w["metric"]["id"] if metric_id is None else metric_id
    return getattr(api.lib, entry)(mid, C.byref(m), C.byref(cam), C.byref(cfg), C.byref(out), None)


BAD = [
    ("metric id", lambda m, c, g: None, 7, api.GP_E_BAD_METRIC),
    ("M < 0", lambda m, c, g: setattr(m, "M", -1.0), None, api.GP_E_BAD_PARAM),
    ("|a| >= M", lambda m, c, g: setattr(m, "a", 1.0), None, api.GP_E_BAD_PARAM),
    ("theta_obs on the axis", lambda m, c, g: setattr(c, "theta_obs", 0.0), None, api.GP_E_BAD_PARAM),
    ("observer inside the capture radius", lambda m, c, g: setattr(c, "r_obs", 1.2), None, api.GP_E_BAD_PARAM),
    ("empty window", lambda m, c, g: setattr(c, "alpha_max", c.alpha_min), None, api.GP_E_BAD_PARAM),
    ("width 0", lambda m, c, g: setattr(c, "width", 0), None, api.GP_E_BAD_PARAM),
    ("rays beyond the image", lambda m, c, g: setattr(c, "ray_begin", 512 * 512 - 10), None, api.GP_E_BAD_PARAM),
    ("stride 0", lambda m, c, g: setattr(c, "ray_stride", 0), None, api.GP_E_BAD_PARAM),
    ("rtol 0", lambda m, c, g: setattr(g, "rtol", 0.0), None, api.GP_E_BAD_PARAM),
    ("scheme 9", lambda m, c, g: setattr(g, "scheme", 9), None, api.GP_E_BAD_PARAM),
    ("r_escape inside r_obs", lambda m, c, g: setattr(g, "r_escape", 10.0), None, api.GP_E_BAD_PARAM),
    ("4 crossings", lambda m, c, g: setattr(g, "max_crossings", 4), None, api.GP_E_BAD_PARAM),
    ("ring with the thin disk", lambda m, c, g: (setattr(g, "ring_half_angle", 0.05), setattr(g, "max_crossings", 1)),
     None, api.GP_E_UNSUPPORTED),
    ("negative ring angle", lambda m, c, g: setattr(g, "ring_half_angle", -1.0), None, api.GP_E_BAD_PARAM),
    ("FP32 with the adaptive scheme", lambda m, c, g: setattr(g, "precision", 1), None, api.GP_E_UNSUPPORTED),
    ("precision 3", lambda m, c, g: setattr(g, "precision", 3), None, api.GP_E_UNSUPPORTED),
    ("mixed precision below its tolerance floor", lambda m, c, g: setattr(g, "precision", 2), None, api.GP_E_BAD_PARAM),
    ("projection 2", lambda m, c, g: setattr(c, "projection", 2), None, api.GP_E_UNSUPPORTED),
    ("screen camera reaching past r_escape", lambda m, c, g: (setattr(c, "projection", 1), setattr(c, "alpha_max", 900.0)),
     None, api.GP_E_BAD_PARAM),
    ("negative focal factor", lambda m, c, g: (setattr(c, "projection", 1), setattr(c, "focal_2f_over_d", -1.0)),
     None, api.GP_E_BAD_PARAM),
    ("segment_steps below -1", lambda m, c, g: setattr(g, "segment_steps", -2), None, api.GP_E_BAD_PARAM),
]


@pytest.mark.parametrize("entry", ["gp_trace", "gp_trace_host", "gp_trace_static"])
@pytest.mark.parametrize("what,mutate,metric_id,code", BAD, ids=[b[0] for b in BAD])
def test_validation_is_synchronous(entry, what, mutate, metric_id, code):
    assert _call(W.workload("C2"), mutate, metric_id, entry=entry) == code


def test_manko_novikov_needs_spin_and_an_explicit_inner_disk_radius():
    w = W.workload("C4")
    assert _call(w, lambda m, c, g: setattr(m, "a", 0.0)) == api.GP_E_BAD_PARAM  # eq 23 divides by S/M
    # no ISCO formula for this metric: disk_r_in = 0 ("use the ISCO") is refused, an explicit one accepted
    assert _call(w, lambda m, c, g: setattr(g, "max_crossings", 2)) == api.GP_E_BAD_PARAM


def test_buffer_checks():
    w = W.workload("C3")
    small = api.gp_out_buffers(C.c_void_p(0x1000), 63 * 128, C.c_void_p(0x2000), 64 * 48, C.c_void_p(0x3000), 64)
    assert _call(w, out=small) == api.GP_E_SIZE
    nodisk = api.gp_out_buffers(C.c_void_p(0x1000), 64 * 128, None, 0, C.c_void_p(0x3000), 64)
    assert _call(w, out=nodisk) == api.GP_E_NULL
    smalldisk = api.gp_out_buffers(C.c_void_p(0x1000), 64 * 128, C.c_void_p(0x2000), 10, C.c_void_p(0x3000), 64)
    assert _call(w, out=smalldisk) == api.GP_E_SIZE
    nocount = api.gp_out_buffers(C.c_void_p(0x1000), 64 * 128, C.c_void_p(0x2000), 64 * 48, None, 0)
    assert _call(w, out=nocount) == api.GP_E_NULL
    misaligned = api.gp_out_buffers(C.c_void_p(0x1008), 64 * 128, C.c_void_p(0x2000), 64 * 48, C.c_void_p(0x3000), 64)
    assert _call(w, out=misaligned) == api.GP_E_BAD_PARAM
    assert api.lib.gp_trace(1, None, None, None, None, None) == api.GP_E_NULL


def test_static_entry_point_limit_and_buffer_checks():
    """gp_trace_static (gp.h): more than GP_STATIC_MAX_RAYS rays are refused with a code of their own before
    any CUDA call is made; the caller's buffers are checked like gp_trace's, except that counters may be NULL."""
    assert gp.gp_static_max_rays() == 1 << 20
    hdr = open(HEADER).read()
    assert re.search(r"#define\s+GP_STATIC_MAX_RAYS\s+1048576\b", hdr) and "GP_E_STATIC_LIMIT = -7" in hdr
    w = W.workload("headline", width=1025, height=1024)
    n = (1 << 20) + 1
    big = api.gp_out_buffers(C.c_void_p(0x1000), n * 128, None, 0, None, 0)
    assert _call(w, lambda m, c, g: setattr(c, "ray_count", n), out=big, entry="gp_trace_static") == api.GP_E_STATIC_LIMIT
    w = W.workload("C3")
    small = api.gp_out_buffers(C.c_void_p(0x1000), 63 * 128, C.c_void_p(0x2000), 64 * 48, None, 0)
    assert _call(w, out=small, entry="gp_trace_static") == api.GP_E_SIZE
    nodisk = api.gp_out_buffers(C.c_void_p(0x1000), 64 * 128, None, 0, None, 0)
    assert _call(w, out=nodisk, entry="gp_trace_static") == api.GP_E_NULL
    misaligned = api.gp_out_buffers(C.c_void_p(0x1008), 64 * 128, C.c_void_p(0x2000), 64 * 48, None, 0)
    assert _call(w, out=misaligned, entry="gp_trace_static") == api.GP_E_BAD_PARAM
    shortcount = api.gp_out_buffers(C.c_void_p(0x1000), 64 * 128, C.c_void_p(0x2000), 64 * 48, C.c_void_p(0x3000), 56)
    assert _call(w, out=shortcount, entry="gp_trace_static") == api.GP_E_SIZE
    oddcount = api.gp_out_buffers(C.c_void_p(0x1000), 64 * 128, C.c_void_p(0x2000), 64 * 48, C.c_void_p(0x3004), 64)
    assert _call(w, out=oddcount, entry="gp_trace_static") == api.GP_E_BAD_PARAM
    assert api.lib.gp_trace_static(1, None, None, None, None, None) == api.GP_E_NULL


def test_static_entry_point_has_no_allocating_call():
    """The body of gp_trace_static, and of the helper that looks up the static array, name no allocation
    routine and no pool; the array is a file-scope `static __device__ __align__(256)` object whose device
    address comes from cudaGetSymbolAddress (in host code its name is only the host-side shadow)."""
    src = open(os.path.join(ROOT, "paper_2310_15183_b200", "csrc", "gp_api.cu")).read()
    assert re.search(r"static __device__ __align__\(256\) unsigned long long g_static_scratch\[", src)
    body = src[src.index("int gp_trace_static("):src.index("int gp_init_conditions(")]
    helper = src[src.index("int static_scratch("):src.index("}  // namespace")]
    body, helper = (re.sub(r"//[^\n]*", "", t) for t in (body, helper))      # code only
    for text in (body, helper):
        for word in ("cudaMalloc", "cudaFree", "scratch_pool", "cudaMemPool", "new ", "malloc(", "std::vector"):
            assert word not in text, word
    assert "cudaGetSymbolAddress(&p, g_static_scratch)" in helper and "GP_CUDA(cudaGetSymbolAddress" in helper
    assert "g_static_scratch" not in body          # host code never passes the shadow to a kernel
    assert "static_scratch(&S)" in body and "P.counters = S;" in body


def _no_gpu():
    try:
        import torch
        return not torch.cuda.is_available()
    except Exception:
        return True


@pytest.mark.skipif(not _no_gpu(), reason="a GPU is present")
def test_no_cpu_fallback_without_a_gpu():
    """Valid arguments on a machine without a GPU: the call reports GP_E_CUDA; nothing is computed."""
    w = W.workload("C2")
    rays = np.zeros(64, dtype=api.RAY_DTYPE)
    out = api.gp_out_buffers(C.c_void_p(rays.ctypes.data), rays.nbytes, None, 0, None, 0)
    assert _call(w, out=out, entry="gp_trace_host") == api.GP_E_CUDA
    assert "CUDA error" in gp.gp_strerror(api.GP_E_CUDA)
    assert not rays.view(np.uint8).any()


def test_shade_and_orbit_validation_is_synchronous():
    """The two entry points of the widened scope validate before anything is enqueued (no GPU needed)."""
    vp = C.c_void_p
    ok = api.shade_struct(dict(width=4, height=4, mode=0))
    call = lambda cfg, rays=0x1000, nb=16 * 128, disk=None, db=0, out=0x2000, ob=64: api.lib.gp_shade(
        C.byref(cfg), vp(rays), nb, vp(disk) if disk else None, db, vp(out), ob, None)
    assert call(api.shade_struct(dict(width=4, height=4, mode=5))) == api.GP_E_BAD_PARAM
    assert call(api.shade_struct(dict(width=0, height=4, mode=0))) == api.GP_E_BAD_PARAM
    assert call(api.shade_struct(dict(width=4, height=4, mode=0, grid_step_deg=-1.0))) == api.GP_E_BAD_PARAM
    assert call(api.shade_struct(dict(width=4, height=4, mode=1, tex_width=0, tex_height=8))) == api.GP_E_BAD_PARAM
    assert call(api.shade_struct(dict(width=4, height=4, mode=2, time_period=0.0))) == api.GP_E_BAD_PARAM
    assert call(api.shade_struct(dict(width=4, height=4, mode=0, disk_overlay=1))) == api.GP_E_NULL
    assert call(api.shade_struct(dict(width=4, height=4, mode=0, disk_overlay=1, g_lo=1.2)), disk=0x3000,
                db=16 * 48) == api.GP_E_BAD_PARAM
    assert call(ok, nb=15 * 128) == api.GP_E_SIZE
    assert call(ok, ob=63) == api.GP_E_SIZE
    assert api.lib.gp_shade(C.byref(ok), None, 0, None, 0, vp(0x2000), 64, None) == api.GP_E_NULL

    m = api.gp_metric_params(1.0, 0.9, 0.0)
    good = dict(rtol=1e-9, atol=1e-9, h0=0.1, h_max=1.0, lambda_end=10.0, n_samples=4)
    orb = lambda cfg, n=2, sb=2 * 4 * 64, stb=8, nsb=16, metric=m, mid=api.GP_KERR: api.lib.gp_integrate_orbits(
        mid, C.byref(metric), C.byref(api.orbit_struct(cfg)), vp(0x1000), n, vp(0x2000), sb, vp(0x3000), stb,
        vp(0x4000), nsb, None)
    for bad in (dict(good, rtol=0.0), dict(good, atol=-1.0), dict(good, h0=0.0), dict(good, h_max=-1.0),
                dict(good, lambda_end=0.0), dict(good, n_samples=0), dict(good, max_steps=-1)):
        assert orb(bad) == api.GP_E_BAD_PARAM, bad
    assert orb(good, sb=2 * 4 * 64 - 1) == api.GP_E_SIZE
    assert orb(good, stb=7) == api.GP_E_SIZE and orb(good, nsb=15) == api.GP_E_SIZE
    assert orb(good, mid=9) == api.GP_E_BAD_METRIC
    assert orb(good, metric=api.gp_metric_params(1.0, 1.5, 0.0)) == api.GP_E_BAD_PARAM
    assert orb(good, n=0) == api.GP_OK            # nothing to do, nothing enqueued
    assert orb(good, n=-1) == api.GP_E_BAD_PARAM


def test_alignment_is_validated_before_anything_is_enqueued():
    """A misaligned caller buffer would raise a sticky misaligned-address fault inside a kernel that uses
    vector loads / stores; every entry point refuses it synchronously instead (GP_E_BAD_PARAM)."""
    vp = C.c_void_p
    ok = api.shade_struct(dict(width=4, height=4, mode=0))
    shade = lambda rays=0x1000, disk=None, out=0x2000, cfg=ok: api.lib.gp_shade(
        C.byref(cfg), vp(rays), 16 * 128, vp(disk) if disk else None, 16 * 48 if disk else 0, vp(out), 64, None)
    assert shade(rays=0x1008) == api.GP_E_BAD_PARAM            # records are read with 128-bit loads
    assert shade(out=0x2002) == api.GP_E_BAD_PARAM             # one 32-bit store per pixel
    ov = api.shade_struct(dict(width=4, height=4, mode=0, disk_overlay=1))
    assert shade(disk=0x3004, cfg=ov) == api.GP_E_BAD_PARAM
    m = api.gp_metric_params(1.0, 0.9, 0.0)
    good = api.orbit_struct(dict(rtol=1e-9, atol=1e-9, h0=0.1, h_max=1.0, lambda_end=10.0, n_samples=4))
    orb = lambda st=0x1000, sa=0x2000, stat=0x3000, ns=0x4000: api.lib.gp_integrate_orbits(
        api.GP_KERR, C.byref(m), C.byref(good), vp(st), 2, vp(sa), 2 * 4 * 64, vp(stat), 8, vp(ns), 16, None)
    assert orb(sa=0x2010) == api.GP_E_BAD_PARAM                # samples: st.global.v4.f64, 32-byte aligned
    assert orb(sa=0x2008) == api.GP_E_BAD_PARAM
    assert orb(st=0x1004) == api.GP_E_BAD_PARAM
    assert orb(stat=0x3002) == api.GP_E_BAD_PARAM
    assert orb(ns=0x4004) == api.GP_E_BAD_PARAM
    # step-level entry points
    w = W.workload("C2")
    cam = api.camera_struct(w["camera"], 0, 8, 1)
    assert api.lib.gp_init_conditions(1, C.byref(m), C.byref(cam), vp(0x1004), 8 * 64, None, 0, None) == api.GP_E_BAD_PARAM
    assert api.lib.gp_init_conditions(1, C.byref(m), C.byref(cam), vp(0x1000), 8 * 64, vp(0x2004), 8 * 16, None) == api.GP_E_BAD_PARAM
    assert api.lib.gp_eval_metric(1, C.byref(m), vp(0x1004), 4, vp(0x2000), 4 * 120, None) == api.GP_E_BAD_PARAM
    assert api.lib.gp_eval_rhs(1, C.byref(m), vp(0x1000), 4, vp(0x2004), 4 * 48, None) == api.GP_E_BAD_PARAM
    # gp_trace: records 32-byte, disk and counters 8-byte
    for out in (api.gp_out_buffers(vp(0x1010), 64 * 128, vp(0x2000), 64 * 48, vp(0x3000), 64),
                api.gp_out_buffers(vp(0x1000), 64 * 128, vp(0x2004), 64 * 48, vp(0x3000), 64),
                api.gp_out_buffers(vp(0x1000), 64 * 128, vp(0x2000), 64 * 48, vp(0x3004), 64)):
        assert _call(W.workload("C3"), out=out) == api.GP_E_BAD_PARAM


def test_no_tuning_hooks_or_process_wide_device_state_in_the_product():
    """The launch path reads no environment variable, and what it caches is keyed by device id."""
    src = open(os.path.join(ROOT, "paper_2310_15183_b200", "csrc", "gp_api.cu")).read()
    assert "getenv" not in src
    assert "static unsigned long long *dcount" not in src and "static cudaMemPool_t pool =" not in src
    assert "cache[kMaxDevices]" in src and "std::mutex" in src
