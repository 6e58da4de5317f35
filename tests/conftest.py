import os
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


@pytest.fixture(scope="session")
def water192():
    """BASELINE.json config 0: 192-atom water box, literal N(0,1/fan_in) weights."""
    import gen
    from gen.weights import MODELS
    from oracle import Oracle
    spec = MODELS["W192"]
    coord, types, box = gen.make_system("W192")
    emb, fit = gen.make_weights(spec)
    return dict(spec=spec, coord=coord, types=types, box=box, emb=emb, fit=fit,
                oracle=Oracle.from_spec(spec, emb, fit))


@pytest.fixture(scope="session")
def water192_cond(water192):
    """Same draw with the fitting W0 scaled by 1/Nm (the 'conditioned' set: no saturated fitting units)."""
    import gen
    from oracle import Oracle
    spec = water192["spec"]
    fit = gen.condition_fit_w0(spec, water192["fit"])
    out = dict(water192)
    out.update(fit=fit, oracle=Oracle.from_spec(spec, water192["emb"], fit))
    return out


def small_model(ntypes=2, s1=4, m_axis=3, fit_width=8, sel=(12, 20), rcut=4.0, rcut_smth=1.0, seed=7,
                fit_scale=0.05):
    """A tiny model (fast brute-force checks); weights drawn like gen.make_weights, fitting W0 damped."""
    import gen
    from gen.weights import ModelSpec
    spec = ModelSpec("tiny", ntypes, rcut, rcut_smth, tuple(sel), s1, m_axis, fit_width, 0)
    emb, fit = gen.make_weights(spec, seed=seed)
    fit = gen.condition_fit_w0(spec, fit, scale=fit_scale)
    return spec, emb, fit


def random_box(n, L, ntypes, seed, min_dist=0.7):
    """n random atoms in a cubic box with a minimum pair distance (rejection sampling); raw coords in [0,L)."""
    rng = np.random.default_rng(seed)
    pts = []
    while len(pts) < n:
        p = rng.uniform(0, L, 3)
        ok = True
        for q in pts:
            d = p - q
            d -= L * np.round(d / L)
            if np.dot(d, d) < min_dist ** 2:
                ok = False
                break
        if ok:
            pts.append(p)
    coord = np.array(pts)
    types = rng.integers(0, ntypes, n).astype(np.int32)
    return coord, types, np.diag([L, L, L]).reshape(9).astype(np.float64)


_ORACLE_FULL = {}


def oracle_full(name, conditioned):
    """The CPU oracle's complete evaluation (dpo_eval over its own cell list, itself pinned against its brute-force search
    in tests/test_oracle_nlist.py) of a BASELINE.json workload at full size, cached for the session: the reference of
    every element-by-element parity test at the sizes bench.py times.  Returns (spec, emb, fit, coord, types, box, ref)."""
    key = (name, bool(conditioned))
    if key not in _ORACLE_FULL:
        import gen
        from gen.weights import MODELS
        from oracle import Oracle
        spec = MODELS[name]
        coord, types, box = gen.make_system(name)
        emb, fit = gen.make_weights(spec)
        if conditioned:
            fit = gen.condition_fit_w0(spec, fit)
        ref = Oracle.from_spec(spec, emb, fit).eval(coord, types, box, cells=True)
        _ORACLE_FULL[key] = (spec, emb, fit, coord, types, box, ref)
    return _ORACLE_FULL[key]


def oracle_forces_of(orc, coord, types, box, atoms):
    """Forces of the listed atoms from the oracle's per-row pieces, for boxes too large for a whole oracle evaluation:
    F_i = sum_k f_ik - sum_{j : i in L(j)} f_{j, slot of i}   (Eq. 10 with ProdForce; the
    assembly is pinned by tests/test_oracle_physics.py::test_atom_rows_pieces_assemble_to_eval).  Needs no neighbour
    overflow (then i in L(j) <=> j in L(i)).  Returns (F [len(atoms)][3], E_i [len(atoms)], nlist rows of the atoms)."""
    atoms = np.asarray(atoms, dtype=np.int64)
    nl_i, ovf = orc.build_nlist(coord, types, box, rows=atoms)
    assert ovf == 0
    nbrs = np.unique(nl_i[nl_i >= 0]).astype(np.int64)
    rows = np.unique(np.concatenate([atoms, nbrs]))
    nl, ovf = orc.build_nlist(coord, types, box, rows=rows)
    assert ovf == 0
    out = orc.atom_rows(coord, types, box, rows, nl)
    where = {int(r): k for k, r in enumerate(rows)}
    F = np.zeros((len(atoms), 3))
    E = np.zeros(len(atoms))
    for a, i in enumerate(atoms):
        qi = where[int(i)]
        F[a] = out["fslot"][qi][nl[qi] >= 0].sum(0)
        E[a] = out["atom_energy"][qi]
        for j in nl[qi][nl[qi] >= 0]:
            qj = where[int(j)]
            hit = np.where(nl[qj] == i)[0]
            assert len(hit) == 1
            F[a] -= out["fslot"][qj, hit[0]]
    return F, E, nl_i
