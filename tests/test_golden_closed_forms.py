"""tests/golden/closed_forms.txt against the oracle and the library's host helpers (no GPU)."""
import math
import os

import pytest

import paper_2310_15183_b200 as gp
from oracle import oracle as O
from paper_2310_15183_b200 import api

HERE = os.path.dirname(os.path.abspath(__file__))


def golden():
    out = {}
    for ln in open(os.path.join(HERE, "golden", "closed_forms.txt")):
        ln = ln.split("#")[0].split()
        if len(ln) == 2:
            out[ln[0]] = float(ln[1])
    return out


def test_golden_values_pin_both_sides():
    g = golden()
    assert len(g) == 12
    for a in ("0.9", "0.998"):
        m = dict(id=1, M=1.0, a=float(a), q=0.0)
        rh, ri = O.radii(m)
        assert rh == pytest.approx(g[f"r_plus_a{a}"], abs=2e-15) and ri == pytest.approx(g[f"r_isco_a{a}"], abs=2e-13)
        rh2, ri2 = gp.gp_metric_radii(gp.GP_KERR, api.gp_metric_params(1.0, float(a), 0.0))
        assert rh2 == pytest.approx(g[f"r_plus_a{a}"], abs=2e-15) and ri2 == pytest.approx(g[f"r_isco_a{a}"], abs=2e-13)
    om, ut, _ = O.kepler(dict(id=1, M=1.0, a=0.998, q=0.0), 6.0, 1.0, 0.0)
    assert om == pytest.approx(g["omega_k_a0.998_r6"], rel=1e-12) and ut == pytest.approx(g["ut_a0.998_r6"], rel=1e-12)
    # closed forms re-evaluated here, independently of both sides
    assert g["b_crit_schwarzschild"] == pytest.approx(3.0 * math.sqrt(3.0), abs=1e-15)
    al = (-1.0 + math.sqrt(1.0 - 0.81)) / 0.9
    k = (1.0 - al * al) / (1.0 + al * al)
    assert al == pytest.approx(g["mn_alpha_a0.9"], abs=1e-15) and k == pytest.approx(g["mn_k_a0.9"], abs=1e-15)
    assert 0.5 / k ** 3 == pytest.approx(g["mn_beta_a0.9_q0.5"], rel=1e-14)
    rh, _ = O.radii(dict(id=2, M=1.0, a=0.9, q=0.5))
    assert rh == pytest.approx(1.0 + g["mn_k_a0.9"], abs=1e-15)
