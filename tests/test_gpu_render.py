"""The frame renderer (trace + image formation + file) — the paper's two scripts through the C-ABI."""
import os
import struct
import zlib

import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def _read_png(path):
    data = open(path, "rb").read()
    assert data[:8] == b"\x89PNG\r\n\x1a\n"
    pos, idat, ihdr = 8, b"", None
    while pos < len(data):
        n, tag = struct.unpack(">I4s", data[pos:pos + 8])
        body = data[pos + 8:pos + 8 + n]
        assert struct.unpack(">I", data[pos + 8 + n:pos + 12 + n])[0] == zlib.crc32(tag + body) & 0xffffffff
        if tag == b"IHDR":
            ihdr = struct.unpack(">IIBBBBB", body)
        if tag == b"IDAT":
            idat += body
        pos += 12 + n
    w, h = ihdr[0], ihdr[1]
    raw = zlib.decompress(idat)
    rows = np.frombuffer(raw, dtype=np.uint8).reshape(h, 1 + 4 * w)
    assert (rows[:, 0] == 0).all()
    return rows[:, 1:].reshape(h, w, 4)


@pytest.mark.parametrize("args", [["--workload", "C2", "--mode", "grid"],
                                  ["--workload", "C3", "--mode", "texture", "--disk", "--supersample", "2"],
                                  ["--workload", "C4", "--mode", "time", "--disk", "--inclination", "80"],
                                  ["--workload", "headline_rk4", "--mode", "grid", "--screen-camera"],
                                  ["--workload", "C3", "--mode", "grid", "--ring", "0.06", "--inclination", "78"]],
                         ids=["kerr_grid", "kerr_disk_texture_ss2", "mn_disk_time", "rk4_screen_camera", "kerr_solid_ring"])
def test_render_writes_an_image(tmp_path, args):
    from paper_2310_15183_b200 import render
    out = str(tmp_path / "frame.png")
    if "C4" in args:
        import gp_workloads as W
        W.WORKLOADS["C4"]["cfg"]["max_steps"] = 2000          # keep the stalled interior short in the test
    try:
        assert render.main(args + ["--size", "96", "--out", out]) == 0
    finally:
        if "C4" in args:
            W.WORKLOADS["C4"]["cfg"]["max_steps"] = 200_000
    img = _read_png(out)
    assert img.shape == (96, 96, 4) and (img[..., 3] == 255).all()
    colours = np.unique(img.reshape(-1, 4), axis=0)
    assert len(colours) >= 4                                   # sky, lines or texture, shadow, ...
    shadow = (img[..., :3] == (0, 255, 255)).all(-1) if "time" in args else (img[..., :3] == 0).all(-1)
    assert 0.005 < shadow.mean() < 0.6                         # there is a shadow, and it is not the whole frame
    ppm = str(tmp_path / "frame.ppm")
    assert render.main(args + ["--size", "32", "--out", ppm]) == 0
    assert open(ppm, "rb").read(2) == b"P6" and os.path.getsize(ppm) == len(b"P6\n32 32\n255\n") + 32 * 32 * 3
