"""The oracle against tests/golden/closed_forms.json: values fixed by mathematics (each entry cites
the formula of the paper or the textbook identity it instantiates), never produced by oracle/ or by
the CUDA path.  The GPU leg (-m gpu) runs the same fixtures through the C ABI."""
import json
import os

import numpy as np
import pytest

import oracle

GOLD = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "closed_forms.json")))


def _cell(c):
    return np.array([[c[0], c[1]], [c[2], c[3]]], dtype=np.float32)


@pytest.mark.parametrize("g", GOLD["bilinear"], ids=lambda g: str(g["value"]))
def test_bilinear_golden(g):
    out = oracle.bilinear(_cell(g["corners"]), oracle.geom(2, 2, 0, 0, 1, 1), oracle.geom(1, 1, g["t"], g["s"], 1, 1))
    assert abs(out[0, 0] - g["value"]) <= 1e-14


@pytest.mark.parametrize("g", GOLD["spline1d"], ids=lambda g: f'{g["z"]}@{g["x"]}')
def test_spline1d_golden(g):
    val, M = oracle.spline1d(g["z"], 1.0, [g["x"]])
    assert abs(val[0] - g["value"]) <= 1e-13
    assert np.abs(M - np.array(g["M"])).max() <= 1e-13


@pytest.mark.parametrize("g", GOLD["spline2d"])
def test_spline2d_golden(g):
    z = np.outer(g["g"], g["f"]).astype(np.float32)
    n = len(g["f"])
    out = oracle.spline(z, oracle.geom(n, n, 0, 0, 1, 1), oracle.geom(1, 1, g["x"], g["y"], 1, 1))
    assert abs(out[0, 0] - g["value"]) <= 1e-13


@pytest.mark.parametrize("g", GOLD["kriging"], ids=lambda g: g["cite"][:24])
def test_kriging_golden(g):
    v = oracle.vgm(g["model"], g["range"], g["sill"], g["nugget"])
    r = oracle.krige_points(g["x"], g["y"], g["z"], [g["xq"]], [g["yq"]], v, len(g["x"]), want_lambda=True)
    lam = r["lam"][0][np.argsort(r["nbr"][0])]                # weights in input order
    assert np.abs(lam - np.array(g["lambda"])).max() <= 2e-7  # fp32 coordinates of the fixture
    assert abs(r["zhat"][0] - g["zhat"]) <= 5e-6


@pytest.mark.gpu
def test_golden_through_the_c_abi():
    import torch
    import paper_2505_22675_b200 as b
    from paper_2505_22675_b200 import workloads as W
    for g in GOLD["bilinear"]:
        out = b.interp_bilinear(torch.from_numpy(_cell(g["corners"])).cuda(), W.Geom(2, 2, 0, 0, 1, 1), W.Geom(1, 1, g["t"], g["s"], 1, 1))
        assert abs(float(out[0, 0]) - g["value"]) <= 1e-6
    for g in GOLD["spline2d"]:
        z = torch.from_numpy(np.outer(g["g"], g["f"]).astype(np.float32)).cuda()
        n = len(g["f"])
        out = b.interp_spline(z, W.Geom(n, n, 0, 0, 1, 1), W.Geom(1, 1, g["x"], g["y"], 1, 1))
        assert abs(float(out[0, 0]) - g["value"]) <= 1e-6
    for g in GOLD["kriging"]:
        x, y, z = (torch.tensor(g[a], dtype=torch.float32, device="cuda") for a in ("x", "y", "z"))
        idx = b.krige_build_index(x, y, z)
        out = b.krige_predict(idx, W.Geom(1, 1, g["xq"], g["yq"], 1, 1), g["model"], g["range"], g["sill"], g["nugget"], len(g["x"]))
        idx.free()
        assert abs(float(out[0, 0]) - g["zhat"]) <= 1e-4
