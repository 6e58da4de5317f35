"""Pins taken from numbers the paper prints (tests/golden/paper_values.txt, each with its citation)."""
import os

import numpy as np

from gen.weights import MODELS, emb_net_size

HERE = os.path.dirname(os.path.abspath(__file__))


def _golden():
    out = {}
    with open(os.path.join(HERE, "golden", "paper_values.txt")) as fh:
        for line in fh:
            line = line.split("#")[0].strip()
            if not line:
                continue
            k, v = line.split("=")
            out[k.strip()] = v.strip()
    return out


def test_model_shapes_follow_the_paper():
    g = _golden()
    w = MODELS["W192"]
    assert w.nm == int(g["water_nm"])
    assert [w.emb_s1, 2 * w.emb_s1, 4 * w.emb_s1] == [int(x) for x in g["emb_widths"].split()]
    assert [w.fit_width] * 3 == [int(x) for x in g["fit_widths"].split()]
    assert w.rcut == float(g["water_rcut"]) and MODELS["Cu32k"].rcut == float(g["copper_rcut"])
    # the O-H embedding batch is (number of O atoms) x sel_H rows INCLUDING padded slots.
    n_o = int(g["matmul_atoms"]) // 3
    assert n_o * w.sel[1] == int(g["matmul_rows"])
    assert w.dim_descrpt == 1600 and MODELS["Cu32k"].dim_descrpt == 2048     # BASELINE.json fitting inputs
    assert emb_net_size(25) == 25 + 25 + 25 * 50 + 50 + 50 * 100 + 100


def test_eq13_memory_example():
    g = _golden()
    gb = float(g["eq13_copies"]) * int(g["eq13_nl"]) * int(g["eq13_nm"]) * int(g["eq13_m"]) * 8 / 1e9
    assert abs(gb - float(g["eq13_gb"])) < 0.005


def test_system_sizes():
    g = _golden()
    assert 192 * 64 * 32 * 32 == int(g["water_atoms"])
    assert 4 * 384 * 384 * 192 == int(g["copper_atoms"])
    import gen
    assert gen.CONFIGS["Cu32k"].box_len == 20 * float(g["fcc_a"])
    c, t, b = gen.make_system("W192")
    assert c.shape == (192, 3) and t.tolist()[:3] == [0, 1, 1] and abs(b[0] - 12.42) < 1e-12
    assert np.all(c >= 0) and np.all(c < 12.42)
