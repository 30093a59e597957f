"""gp_trace_static (include/gp.h): the trace for callers that may not allocate.  Its scratch — the work
counter, the totals, and the slot lists of segmented tracing — is the library's file-scope static device
array instead of caller memory and the stream-ordered pool, so a call makes no cudaMalloc at all; at most
GP_STATIC_MAX_RAYS rays per call.

The kernels are the ones gp_trace launches and a ray's arithmetic does not depend on which lane draws it,
so the bar is the one the repository uses wherever the same kernel runs twice (segmented tracing, shards,
host path): records identical BIT FOR BIT, and the totals equal.  Every case makes two static calls in a
row, the second on top of whatever the first left in the array.

Collected last on purpose (pytest -x must not lose the parity tests behind a failure
here); passes alone in a fresh process and after the rest of the suite (nothing here depends on, or
leaves behind, state that another test reads: the array is cleared by every call that uses it).
"""
import ctypes as C
import math

import numpy as np
import pytest

import gp_workloads as W

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def gp():
    import paper_2310_15183_b200 as gp
    return gp


def _static(gp, w, with_counters=True):
    """gp_trace_static on a workload; returns (rays, disk, counters) like api.trace_workload.  The caller's
    buffers are filled with a byte pattern first so that an element the kernel failed to write shows."""
    import torch
    api = gp.api
    cam = api.camera_struct(w["camera"])
    cfg = api.cfg_struct(w["cfg"])
    n = cam.ray_count
    rays = torch.full((max(n, 1) * 128,), 0xA5, dtype=torch.uint8, device="cuda")
    need_disk = cfg.max_crossings > 0 or cfg.ring_half_angle > 0.0
    disk = torch.full((max(n, 1) * 48,), 0xA5, dtype=torch.uint8, device="cuda") if need_disk else None
    counters = torch.full((64,), 0xA5, dtype=torch.uint8, device="cuda") if with_counters else None
    gp.gp_trace_static(w["metric"]["id"], api.metric_struct(w["metric"]), cam, cfg, rays, disk, counters)
    torch.cuda.current_stream().synchronize()
    r = rays.cpu().numpy().view(api.RAY_DTYPE)[:n]
    d = disk.cpu().numpy().view(api.DISK_DTYPE)[:n] if disk is not None else None
    c = counters.cpu().numpy().view("<u8") if with_counters else None
    return r, d, c


def _same(a, b, label):
    rays, disk, counters = a
    ref_rays, ref_disk, ref_counters = b
    assert len(rays) == len(ref_rays), label
    assert rays.tobytes() == ref_rays.tobytes(), f"{label}: ray records differ"
    assert (disk is None) == (ref_disk is None), label
    if disk is not None:
        assert disk.tobytes() == ref_disk.tobytes(), f"{label}: disk records differ"
    if counters is not None:
        # [1] rays finished, [2] attempted steps, [3] RHS evaluations; [0] >= ray_count at exit
        assert np.array_equal(counters[1:4], ref_counters[1:4]), (label, counters, ref_counters)
        assert counters[6] == ref_counters[6] and counters[7] >= counters[4] > 0


def _cases():
    kerr_disk = W.workload("C3", width=320, height=200)                       # adaptive, thin disk, ragged tail
    kerr = W.workload("C2", width=300, height=300)                            # adaptive, no object
    rk4 = W.workload("C5a", width=257, height=131)                            # fixed step, odd sizes
    mn = W.workload("C4", width=192, height=192, theta_obs=math.radians(82.0))
    mn["cfg"].update(max_steps=30000, segment_steps=2500)                     # 12 rounds through the static lists
    mn_ring = W.workload("C4", width=160, height=160, theta_obs=math.radians(82.0))
    mn_ring["cfg"].update(max_steps=600, segment_steps=7, ring_half_angle=0.05, disk_r_in=5.0, disk_r_out=14.0)
    small = W.workload("C1", width=33, height=3)                              # 99 rays: less than one block
    return [("kerr_disk", kerr_disk), ("kerr", kerr), ("rk4", rk4), ("mn_segmented", mn), ("mn_ring_86_rounds", mn_ring),
            ("small", small)]


def test_static_scratch_matches_gp_trace_on_two_calls_in_a_row(gp):
    """Each workload: the existing path once, the static path twice in a row; then the workloads
    interleaved, so that every call starts from the array as a DIFFERENT kind of call left it (a larger
    image's work counter, a segmented call's list counts and lists)."""
    cases = _cases()
    ref = {}
    for name, w in cases:
        ref[name] = gp.api.trace_workload(w)
        assert ref[name][2][1] == len(ref[name][0]) > 0
        first = _static(gp, w)
        second = _static(gp, w)
        _same(first, ref[name], f"{name}, first call")
        _same(second, ref[name], f"{name}, second call")
    for name, w in cases[::-1] + cases[1::2]:
        _same(_static(gp, w), ref[name], f"{name}, interleaved")
    # the existing path is untouched by what the static calls left behind
    name, w = cases[0]
    _same(gp.api.trace_workload(w), ref[name], "gp_trace after the static calls")


def test_static_scratch_back_to_back_without_a_host_sync(gp):
    """Two static calls enqueued on one stream with no synchronisation between them: stream order alone
    keeps the second call's memset behind the first call's kernel."""
    import torch
    api = gp.api
    wa = W.workload("C3", width=256, height=256)
    wb = W.workload("C5a", width=200, height=100)
    bufs = []
    for w in (wa, wb, wa):
        cam, cfg = api.camera_struct(w["camera"]), api.cfg_struct(w["cfg"])
        rays = torch.empty(cam.ray_count * 128, dtype=torch.uint8, device="cuda")
        disk = torch.empty(cam.ray_count * 48, dtype=torch.uint8, device="cuda") if cfg.max_crossings > 0 else None
        cnt = torch.empty(64, dtype=torch.uint8, device="cuda")
        bufs.append((w, cam, cfg, rays, disk, cnt))
    for w, cam, cfg, rays, disk, cnt in bufs:       # all three enqueued before anything is waited for
        gp.gp_trace_static(w["metric"]["id"], api.metric_struct(w["metric"]), cam, cfg, rays, disk, cnt)
    torch.cuda.synchronize()
    for w, cam, cfg, rays, disk, cnt in bufs:
        got = (rays.cpu().numpy().view(api.RAY_DTYPE),
               disk.cpu().numpy().view(api.DISK_DTYPE) if disk is not None else None,
               cnt.cpu().numpy().view("<u8"))
        _same(got, api.trace_workload(w), "enqueued back to back")


def test_static_scratch_at_its_limit_and_beyond(gp):
    """ray_count == GP_STATIC_MAX_RAYS (the 1024 x 1024 headline image) runs and matches gp_trace; one ray
    more is refused with GP_E_STATIC_LIMIT before anything is enqueued, and the message names the limit."""
    import torch
    api = gp.api
    limit = gp.gp_static_max_rays()
    assert limit == 1 << 20
    w = W.workload("headline")
    assert W.n_rays(w) == limit
    ref = api.trace_workload(w)
    _same(_static(gp, w), ref, "headline, first call")
    _same(_static(gp, w, with_counters=False), ref, "headline, second call, no counters asked for")

    big = W.workload("headline", width=1025, height=1024)
    cam, cfg = api.camera_struct(big["camera"], 0, limit + 1, 1), api.cfg_struct(big["cfg"])
    rays = torch.full(((limit + 1) * 128,), 0x5A, dtype=torch.uint8, device="cuda")
    with pytest.raises(api.GpError) as err:
        gp.gp_trace_static(big["metric"]["id"], api.metric_struct(big["metric"]), cam, cfg, rays, None, None)
    assert err.value.code == api.GP_E_STATIC_LIMIT
    assert "1048576" in str(err.value) and "GP_STATIC_MAX_RAYS" in str(err.value)
    torch.cuda.synchronize()
    assert int(rays.min()) == 0x5A == int(rays.max()), "a refused call wrote to the caller's buffer"
    # the same image in two tiles of at most `limit` rays each, as gp.h suggests
    total = W.n_rays(big)
    whole = api.trace_workload(big)
    parts = []
    for begin in range(0, total, limit):
        count = min(limit, total - begin)
        cam = api.camera_struct(big["camera"], begin, count, 1)
        r = torch.empty(count * 128, dtype=torch.uint8, device="cuda")
        gp.gp_trace_static(big["metric"]["id"], api.metric_struct(big["metric"]), cam, cfg, r, None, None)
        parts.append(r.cpu().numpy())
    assert len(parts) == 2 and b"".join(p.tobytes() for p in parts) == whole[0].tobytes()


def test_static_entry_point_allocates_nothing(gp):
    """Device memory in use (driver view, cudaMemGetInfo) does not move across static calls once the first
    one has loaded the kernels, and torch's allocator is not involved either."""
    import torch
    api = gp.api
    w = W.workload("C4", width=128, height=128, theta_obs=math.radians(82.0))
    w["cfg"].update(max_steps=20000, segment_steps=2000)      # the variant whose gp_trace path allocates lists
    cam, cfg = api.camera_struct(w["camera"]), api.cfg_struct(w["cfg"])
    rays = torch.empty(cam.ray_count * 128, dtype=torch.uint8, device="cuda")
    m = api.metric_struct(w["metric"])
    gp.gp_trace_static(w["metric"]["id"], m, cam, cfg, rays, None, None)     # module load, occupancy query
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    reserved0 = torch.cuda.memory_reserved()
    for _ in range(3):
        gp.gp_trace_static(w["metric"]["id"], m, cam, cfg, rays, None, None)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 >= free0 and torch.cuda.memory_reserved() == reserved0
    assert rays.cpu().numpy().view(api.RAY_DTYPE).tobytes() == api.trace_workload(w)[0].tobytes()


def test_static_entry_point_validates_like_gp_trace(gp):
    """Same synchronous validation as gp_trace: bad configuration, missing / short / misaligned buffers."""
    import torch
    api = gp.api
    w = W.workload("C3", width=16, height=16)
    cam, cfg, m = api.camera_struct(w["camera"]), api.cfg_struct(w["cfg"]), api.metric_struct(w["metric"])
    rays = torch.empty(256 * 128 + 32, dtype=torch.uint8, device="cuda")
    disk = torch.empty(256 * 48, dtype=torch.uint8, device="cuda")
    cnt = torch.empty(72, dtype=torch.uint8, device="cuda")

    def code(*a):
        with pytest.raises(api.GpError) as err:
            gp.gp_trace_static(w["metric"]["id"], m, cam, cfg, *a)
        return err.value.code

    assert code(rays[:256 * 128 - 1], disk, None) == api.GP_E_SIZE
    assert code(rays[:256 * 128], disk[:100], None) == api.GP_E_SIZE
    assert code(rays[:256 * 128], None, None) == api.GP_E_NULL
    assert code(rays[8:8 + 256 * 128], disk, None) == api.GP_E_BAD_PARAM          # rays not 32-byte aligned
    assert code(rays[:256 * 128], disk, cnt[:63]) == api.GP_E_SIZE
    assert code(rays[:256 * 128], disk, cnt[4:68]) == api.GP_E_BAD_PARAM          # counters not 8-byte aligned
    bad = api.cfg_struct(dict(w["cfg"], rtol=-1.0))
    with pytest.raises(api.GpError) as err:
        gp.gp_trace_static(w["metric"]["id"], m, cam, bad, rays[:256 * 128], disk, None)
    assert err.value.code == api.GP_E_BAD_PARAM
    assert api.lib.gp_trace_static(1, C.byref(m), C.byref(cam), C.byref(cfg), None, None) == api.GP_E_NULL
    # and an empty selection is a no-op that still reports zeroed totals
    cam0 = api.camera_struct(w["camera"], 0, 0, 1)
    cnt64 = torch.full((64,), 0xA5, dtype=torch.uint8, device="cuda")
    gp.gp_trace_static(w["metric"]["id"], m, cam0, cfg, None, None, cnt64)
    torch.cuda.synchronize()
    assert not cnt64.cpu().numpy().any()
