"""Pins for the oracle's neighbour search and Alg. 1 formatting.

Nothing here calls the CUDA path.  The pins are facts fixed by geometry (FCC shells, water geometry), by the
definition (symmetry of L(i), section order, padding), and an independent numpy brute force.
"""
import numpy as np
import pytest

import gen
from gen.weights import MODELS, ModelSpec
from oracle import Oracle

from conftest import small_model, random_box


def _oracle(spec):
    emb, fit = gen.make_weights(spec, seed=1)
    return Oracle.from_spec(spec, emb, fit)


def test_fcc_shells_176_neighbours():
    """Perfect FCC a=3.634 A, r_c=8 A: every atom has 12+6+24+12+24+8+48+6+36 = 176 neighbours (lattice
    geometry; next shell at a*sqrt(5)=8.126 A), in ascending distance order."""
    spec = MODELS["Cu32k"]
    coord, types, box = gen.copper_box(6, 0.0, seed=0)          # 864 atoms, L = 21.8 > 2 r_c
    nl, ovf = _oracle(spec).build_nlist(coord, types, box)
    assert ovf == 0
    cnt = (nl >= 0).sum(1)
    assert np.all(cnt == 176)
    a = 3.634
    shells = [(12, 0.5), (6, 1.0), (24, 1.5), (12, 2.0), (24, 2.5), (8, 3.0), (48, 3.5), (6, 4.0), (36, 4.5)]
    L = box[0]
    for i in (0, 17, 500):
        d = coord[nl[i, :176]] - coord[i]
        d -= L * np.round(d / L)
        r = np.linalg.norm(d, axis=1)
        k = 0
        for n, f in shells:
            assert np.allclose(r[k:k + n], a * np.sqrt(f), atol=1e-9)
            k += n
        assert np.all(nl[i, 176:] == -1)


def test_equal_distance_ties_break_by_index():
    """same type and distance -> smaller atom index first.  A simple cubic lattice with
    exactly representable coordinates gives exactly equal distances."""
    n = 6
    g = np.stack(np.meshgrid(*[np.arange(n)] * 3, indexing="ij"), -1).reshape(-1, 3).astype(np.float64) * 2.0
    types = np.zeros(len(g), dtype=np.int32)
    box = np.diag([2.0 * n] * 3).reshape(9)
    spec = ModelSpec("sc", 1, 4.5, 1.0, (64,), 4, 2, 8, 0)
    nl, ovf = _oracle(spec).build_nlist(g, types, box)
    assert ovf == 0
    L = box[0]
    for i in (0, 43, 215):
        js = nl[i][nl[i] >= 0]
        d = g[js] - g[i]
        d -= L * np.round(d / L)
        r2 = (d * d).sum(1)                   # exact small integers
        assert len(js) == 6 + 12 + 8 + 6 + 24   # shells r^2 = 4, 8, 12, 16, 20 (sqrt(20) = 4.47 < 4.5 < sqrt(24))
        assert np.all(np.diff(r2) >= 0)
        for v in np.unique(r2):
            grp = js[r2 == v]
            assert np.all(np.diff(grp) > 0), "ties must be in ascending atom index"


def test_water_geometry_and_sections(water192):
    o, spec = water192["oracle"], water192["spec"]
    coord, types, box = water192["coord"], water192["types"], water192["box"]
    nl, ovf = o.build_nlist(coord, types, box)
    assert ovf == 0 and nl.shape == (192, 138)
    L = box[0]
    sel_o, sel_h = spec.sel
    for i in range(192):
        row = nl[i]
        for lo, hi, t in ((0, sel_o, 0), (sel_o, sel_o + sel_h, 1)):
            sec = row[lo:hi]
            real = sec[sec >= 0]
            assert np.all(sec[:len(real)] >= 0) and np.all(sec[len(real):] == -1)   # -1 only at section tails
            assert np.all(types[real] == t)                                        # sorted by type first
            d = coord[real] - coord[i]
            d -= L * np.round(d / L)
            r = np.linalg.norm(d, axis=1)
            assert np.all(np.diff(r) >= 0) and np.all(r <= spec.rcut)               # then by distance
            assert i not in real
        if types[i] == 0:      # an O atom: its two own H (index i+1, i+2) are the nearest H-section entries
            assert set(row[sel_o:sel_o + 2].tolist()) == {i + 1, i + 2}
            d = coord[row[sel_o:sel_o + 2]] - coord[i]
            d -= L * np.round(d / L)
            assert np.all(np.abs(np.linalg.norm(d, axis=1) - 0.96) < 0.6)           # 0.96 A +- jitter
    # j in L(i)  <=>  i in L(j)
    pairs = {(i, int(j)) for i in range(192) for j in nl[i] if j >= 0}
    assert all((j, i) in pairs for (i, j) in pairs)
    # SURVEY.md probe: ~85 real neighbours per atom at this density and cutoff
    assert 80 < (nl >= 0).sum(1).mean() < 92


def test_against_independent_numpy_bruteforce():
    """Brute force on a small random box, written independently (numpy, round-based minimum image)."""
    spec, emb, fit = small_model()
    coord, types, box = random_box(150, 9.0, 2, seed=3)
    coord = coord + np.array([13.0, -9.0, 4.5])          # raw coordinates outside [0, L) are legal input
    nl, ovf = Oracle.from_spec(spec, emb, fit).build_nlist(coord, types, box)
    L = box[0]
    exp_ovf = 0
    for i in range(len(coord)):
        d = coord - coord[i]
        d -= L * np.round(d / L)
        r = np.sqrt((d * d).sum(1))
        k0 = 0
        for t in range(spec.ntypes):
            idx = np.where((r <= spec.rcut) & (types == t) & (np.arange(len(coord)) != i))[0]
            idx = idx[np.lexsort((idx, r[idx]))]
            exp_ovf += max(0, len(idx) - spec.sel[t])
            idx = idx[:spec.sel[t]]
            exp = np.full(spec.sel[t], -1)
            exp[:len(idx)] = idx
            assert np.array_equal(nl[i, k0:k0 + spec.sel[t]], exp)
            k0 += spec.sel[t]
    assert ovf == exp_ovf


def test_overflow_keeps_nearest_and_counts_drops():
    spec, emb, fit = small_model(sel=(3, 4))
    coord, types, box = random_box(120, 9.0, 2, seed=5)
    big_spec, _, _ = small_model(sel=(60, 60))
    nl_small, ovf = Oracle.from_spec(spec, emb, fit).build_nlist(coord, types, box)
    nl_big, ovf_big = Oracle.from_spec(big_spec, emb, fit).build_nlist(coord, types, box)
    assert ovf_big == 0 and ovf > 0
    assert np.array_equal(nl_small[:, :3], nl_big[:, :3])
    assert np.array_equal(nl_small[:, 3:7], nl_big[:, 60:64])
    assert ovf == int(np.maximum((nl_big[:, :60] >= 0).sum(1) - 3, 0).sum()
                      + np.maximum((nl_big[:, 60:] >= 0).sum(1) - 4, 0).sum())


@pytest.mark.parametrize("name", ["W192", "cu6", "rand"])
def test_cell_list_equals_bruteforce(name, water192):
    if name == "W192":
        o, coord, types, box = water192["oracle"], water192["coord"], water192["types"], water192["box"]
    elif name == "cu6":
        coord, types, box = gen.copper_box(7, 0.05, seed=11)
        o = _oracle(MODELS["Cu32k"])
    else:
        spec, emb, fit = small_model(rcut=2.9)
        coord, types, box = random_box(400, 12.0, 2, seed=9)       # 4 cells per dimension
        coord = coord - 20.0
        o = Oracle.from_spec(spec, emb, fit)
    a, ovf_a = o.build_nlist(coord, types, box)
    b, ovf_b = o.build_nlist(coord, types, box, cells=True)
    assert np.array_equal(a, b) and ovf_a == ovf_b


def test_rows_subset_matches_full(water192):
    o = water192["oracle"]
    full, _ = o.build_nlist(water192["coord"], water192["types"], water192["box"])
    rows = np.array([5, 0, 191, 77])
    sub, _ = o.build_nlist(water192["coord"], water192["types"], water192["box"], rows=rows)
    assert np.array_equal(sub, full[rows])


def test_box_errors(water192):
    from oracle.dpo import OracleError
    o = water192["oracle"]
    bad = water192["box"].copy()
    bad[0] = 11.9                                 # r_c = 6 >= L/2
    with pytest.raises(OracleError):
        o.build_nlist(water192["coord"], water192["types"], bad)
    tri = water192["box"].copy()
    tri[1] = 0.5                                  # not orthorhombic
    with pytest.raises(OracleError):
        o.build_nlist(water192["coord"], water192["types"], tri)
