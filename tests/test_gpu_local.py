"""GPU parity tests of dpb_eval_local (one sub-region with explicit ghost atoms, no box; SURVEY.md §8(e) / §8(f) NEXT
#2, #3) against the oracle's dpo_eval_local, through the C ABI.  Bars as for dpb_eval: the neighbour
list bit-exact; fp64: 1e-10 relative on E, 1e-9 eV/A on F (local AND ghost atoms); mixed precision: 1e-5 / 1e-3.
The ghost shells are built by brute force over the 27 periodic images (tests/test_oracle_local.py)."""
import numpy as np
import pytest

import gen
from gen.weights import MODELS

from conftest import small_model, random_box
from test_oracle_local import brute_force_domain, bricks

pytestmark = pytest.mark.gpu


def _torch():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device (the library has no CPU fallback)")
    return torch


def _bars(precision):
    from paper_2004_11658_b200.binding import FP64
    return (1e-10, 1e-9, 1e-10) if precision == FP64 else (1e-5, 1e-3, 1e-5)


def _gpu_local(m, x, t, nloc, bounds):
    torch = _torch()
    out = m.eval_local(torch.tensor(x, device="cuda"), torch.tensor(t.astype(np.int32), device="cuda"), nloc, bounds,
                       want_nlist=True)
    torch.cuda.synchronize()
    return {k: (v.cpu().numpy() if hasattr(v, "cpu") else v) for k, v in out.items()}


def _domain(coord, types, box, lo, hi, rc):
    loc, own, gxyz, w = brute_force_domain(coord, box, lo, hi, rc)
    x = np.ascontiguousarray(np.concatenate([w[loc], gxyz]))
    t = np.concatenate([types[loc], types[own]]).astype(np.int32)
    bounds = np.concatenate([lo - rc, hi + rc])
    return loc, own, x, t, bounds


def _check(ref, got, precision):
    e_rel, f_abs, v_rel = _bars(precision)
    assert np.array_equal(got["nlist"], ref["nlist"]), "nlist must be bit-exact"
    assert abs(got["energy"][0] - ref["energy"]) <= e_rel * abs(ref["energy"])
    assert np.abs(got["atom_energy"] - ref["atom_energy"]).max() <= e_rel * np.abs(ref["atom_energy"]).max()
    assert np.abs(got["force"] - ref["force"]).max() <= f_abs
    assert np.abs(got["virial"] - ref["virial"]).max() <= v_rel * max(1.0, np.abs(ref["virial"]).max())


@pytest.mark.parametrize("precision_name", ["FP64", "TF32"])
@pytest.mark.parametrize("grid", [(2, 1, 1), (2, 2, 2)])
def test_water192_subregions_against_the_oracle(precision_name, grid):
    """BASELINE config 0 (W192, conditioned weights) cut into bricks: every brick, every output element, ghost forces
    included; then the partition identity against dpb_eval on the periodic box."""
    import paper_2004_11658_b200 as pk
    from oracle import Oracle
    torch = _torch()
    from paper_2004_11658_b200 import binding
    precision = getattr(binding, precision_name)
    spec = MODELS["W192"]
    coord, types, box = gen.make_system("W192")
    emb, fit = gen.make_weights(spec)
    fit = gen.condition_fit_w0(spec, fit)
    orc = Oracle.from_spec(spec, emb, fit)
    m = pk.DPModel.from_spec(spec, emb, fit, precision=precision)
    n = len(coord)
    E, F, V = 0.0, np.zeros((n, 3)), np.zeros((3, 3))
    for lo, hi in bricks(box, grid):
        loc, own, x, t, bounds = _domain(coord, types, box, lo, hi, spec.rcut)
        ref = orc.eval_local(x, t, len(loc))
        got = _gpu_local(m, x, t, len(loc), bounds)
        assert got["force"].shape == (len(x), 3) and np.abs(ref["force"][len(loc):]).max() > 1e-3
        _check(ref, got, precision)
        E += got["energy"][0]
        V += got["virial"]
        np.add.at(F, np.concatenate([loc, own]), got["force"])
    per = m.eval(torch.tensor(coord, device="cuda"), torch.tensor(types, device="cuda"), box)
    torch.cuda.synchronize()
    e_rel, f_abs, v_rel = _bars(precision)
    assert abs(E - per["energy"].item()) <= 2 * e_rel * abs(E)
    assert np.abs(F - per["force"].cpu().numpy()).max() <= 2 * f_abs
    assert np.abs(V - per["virial"].cpu().numpy()).max() <= 2 * v_rel * max(1.0, np.abs(V).max())


def test_cutoff_beyond_half_the_box():
    """r_c >= L/2 (refused by dpb_eval: DPB_EBOX) through explicit images, the paper's formulation:
    one brick = the whole box, every ghost a periodic image; an atom then sees several images of the same neighbour."""
    import paper_2004_11658_b200 as pk
    from oracle import Oracle
    torch = _torch()
    spec, emb, fit = small_model(ntypes=2, s1=8, m_axis=4, fit_width=16, sel=(40, 60), rcut=4.0, rcut_smth=1.0, seed=5,
                                 fit_scale=0.05)
    coord, types, box = random_box(30, 6.5, 2, seed=11, min_dist=1.2)         # L = 6.5 < 2 r_c
    orc = Oracle.from_spec(spec, emb, fit)
    m = pk.DPModel.from_spec(spec, emb, fit)
    with pytest.raises(pk.DPBError):
        m.eval(torch.tensor(coord, device="cuda"), torch.tensor(types, device="cuda"), box)
    lo, hi = np.zeros(3), np.array([box[0], box[4], box[8]])
    loc, own, x, t, bounds = _domain(coord, types, box, lo, hi, spec.rcut)
    assert len(loc) == 30 and len(own) > 60
    ref = orc.eval_local(x, t, 30)
    ids = np.concatenate([loc, own])
    row = ref["nlist"][0]
    owners = ids[row[row >= 0]]
    assert len(set(owners)) < len(owners)                                    # the same atom twice, as two images
    got = _gpu_local(m, x, t, 30, bounds)
    _check(ref, got, 0)


def test_isolated_cluster_and_degenerate_cases():
    import paper_2004_11658_b200 as pk
    from oracle import Oracle
    spec, emb, fit = small_model(ntypes=2, s1=8, m_axis=4, fit_width=16, sel=(30, 40), rcut=4.0, rcut_smth=1.0, seed=6,
                                 fit_scale=0.05)
    coord, types, box = random_box(50, 9.0, 2, seed=3, min_dist=1.2)
    orc = Oracle.from_spec(spec, emb, fit)
    m = pk.DPModel.from_spec(spec, emb, fit)
    x = coord - 200.0                                                         # negative coordinates, far from the origin
    bounds = np.concatenate([x.min(axis=0), x.max(axis=0)])                   # tight: atoms sit ON the bounds
    ref = orc.eval_local(x, types, 50)
    got = _gpu_local(m, x, types, 50, bounds)
    _check(ref, got, 0)
    assert np.abs(got["force"].sum(axis=0)).max() < 1e-9
    # ghosts only
    got0 = _gpu_local(m, x, types, 0, bounds)
    assert got0["energy"][0] == 0.0 and not got0["force"].any() and not got0["virial"].any()
    # a lone atom, and nothing at all
    one = _gpu_local(m, x[:1], types[:1], 1, np.concatenate([x[0], x[0]]))
    ref1 = orc.eval_local(x[:1], types[:1], 1)
    assert abs(one["energy"][0] - ref1["energy"]) <= 1e-10 * max(1.0, abs(ref1["energy"])) and not one["force"].any()
    none = _gpu_local(m, x[:0], types[:0], 0, np.zeros(6))
    assert none["energy"][0] == 0.0
    # an atom outside the bounds is reported, not silently mis-binned
    bad = bounds.copy()
    bad[3] -= 1.0
    with pytest.raises(pk.DPBError):
        _gpu_local(m, x, types, 50, bad)
    # the same degenerate cases with the deterministic reduction
    m.set_deterministic(True)
    _check(ref, _gpu_local(m, x, types, 50, bounds), 0)
    got0 = _gpu_local(m, x, types, 0, bounds)
    assert got0["energy"][0] == 0.0 and not got0["force"].any() and not got0["virial"].any()
    one = _gpu_local(m, x[:1], types[:1], 1, np.concatenate([x[0], x[0]]))
    assert abs(one["energy"][0] - ref1["energy"]) <= 1e-10 * max(1.0, abs(ref1["energy"])) and not one["force"].any()
    m.set_deterministic(False)


@pytest.mark.parametrize("chunk", [0, 40])
def test_deterministic_reduction_in_subregions(chunk):
    """Deterministic reduction + per-atom virial in sub-region mode (the ghosts' lists are built too and name, by the
    list symmetry, the local atoms that push on each ghost): W192 in 2 x 2 x 2 bricks against the oracle's
    dpo_eval_local, ghost forces included; two runs agree bit for bit; the per-atom virial of a brick's local atoms
    equals the periodic box's dpo_atom_virial of the same atoms and sums to the brick's virial.  chunk = 40: local and
    ghost rows in several chunks."""
    import paper_2004_11658_b200 as pk
    from oracle import Oracle
    torch = _torch()
    spec = MODELS["W192"]
    coord, types, box = gen.make_system("W192")
    emb, fit = gen.make_weights(spec)
    fit = gen.condition_fit_w0(spec, fit)
    orc = Oracle.from_spec(spec, emb, fit)
    av_ref = orc.atom_virial(coord, types, box)
    m = pk.DPModel.from_spec(spec, emb, fit)
    if chunk:
        m.set_chunk(chunk)
    m.set_deterministic(True)
    for lo, hi in bricks(box, (2, 2, 2)):
        loc, own, x, t, bounds = _domain(coord, types, box, lo, hi, spec.rcut)
        nloc = len(loc)
        ref = orc.eval_local(x, t, nloc)
        av = torch.full((len(x), 9), float("nan"), dtype=torch.float64, device="cuda")
        m.set_atom_virial(av)
        got = _gpu_local(m, x, t, nloc, bounds)
        _check(ref, got, 0)
        avh = av.cpu().numpy()
        assert np.isnan(avh[nloc:]).all(), "only the local atoms' rows are written"
        scale = max(1.0, np.abs(av_ref).max())
        assert np.abs(avh[:nloc].reshape(-1, 3, 3) - av_ref[loc].reshape(-1, 3, 3)).max() <= 1e-10 * scale
        assert np.abs(avh[:nloc].sum(axis=0).reshape(3, 3) - got["virial"]).max() <= 1e-10 * scale
        again = _gpu_local(m, x, t, nloc, bounds)
        for k in ("energy", "atom_energy", "force", "virial"):
            assert np.array_equal(got[k], again[k]), k
        m.set_atom_virial(None)
    m.set_deterministic(False)


def test_water24k_slab_identity():
    """BASELINE configs[1] (W24k) cut into 2 x 2 x 1 bricks in the launch configuration bench.py uses (default chunk,
    fp64): ghost shells from the 27 images, sum over the bricks against dpb_eval on the periodic box, and a sample of
    local atoms of one brick against the oracle (nlist rows, E_i)."""
    import paper_2004_11658_b200 as pk
    from oracle import Oracle
    torch = _torch()
    spec = MODELS["W24k"]
    coord, types, box = gen.make_system("W24k")
    emb, fit = gen.make_weights(spec)
    fit = gen.condition_fit_w0(spec, fit)
    m = pk.DPModel.from_spec(spec, emb, fit)
    n = len(coord)
    E, F, V = 0.0, np.zeros((n, 3)), np.zeros((3, 3))
    first = None
    for lo, hi in bricks(box, (2, 2, 1)):
        loc, own, x, t, bounds = _domain(coord, types, box, lo, hi, spec.rcut)
        got = _gpu_local(m, x, t, len(loc), bounds)
        if first is None:
            first = (loc, own, x, t, got)
        E += got["energy"][0]
        V += got["virial"]
        np.add.at(F, np.concatenate([loc, own]), got["force"])
    per = m.eval(torch.tensor(coord, device="cuda"), torch.tensor(types, device="cuda"), box)
    torch.cuda.synchronize()
    assert abs(E - per["energy"].item()) <= 1e-10 * abs(E)
    assert np.abs(F - per["force"].cpu().numpy()).max() <= 2e-9
    assert np.abs(V - per["virial"].cpu().numpy()).max() <= 1e-10 * max(1.0, np.abs(V).max())
    loc, own, x, t, got = first
    orc = Oracle.from_spec(spec, emb, fit)
    rows = np.random.default_rng(5).choice(len(loc), size=48, replace=False).astype(np.int64)
    big = np.diag([1e300] * 3).reshape(-1)                                    # the oracle's open-boundary box
    nl = orc.build_nlist(x, t, big, rows=rows)
    nl = nl[0] if isinstance(nl, tuple) else nl
    assert np.array_equal(got["nlist"][rows], nl)
    ar = orc.atom_rows(x, t, big, rows, nl)
    assert np.abs(got["atom_energy"][rows] - ar["atom_energy"]).max() <= 1e-10 * np.abs(ar["atom_energy"]).max()


@pytest.mark.parametrize("name", ["W192", "W24k"])
def test_decomposition_driver_on_one_gpu(name):
    """paper_2004_11658_b200.dd with world size 1 on the device: the forward exchange makes the periodic images, the
    reverse exchange folds their forces back, dpb_eval_local does the arithmetic; against dpb_eval on the same box.
    (The multi-rank routes are covered over gloo in tests/test_dd_gloo.py.)"""
    import paper_2004_11658_b200 as pk
    from paper_2004_11658_b200.dd import BrickDecomposition
    torch = _torch()
    spec = MODELS[name]
    coord, types, box = gen.make_system(name)
    emb, fit = gen.make_weights(spec)
    fit = gen.condition_fit_w0(spec, fit)
    m = pk.DPModel.from_spec(spec, emb, fit)
    dc, dt = torch.tensor(coord, device="cuda"), torch.tensor(types, device="cuda")
    per = m.eval(dc, dt, box)
    dd = BrickDecomposition(box, spec.rcut, grid=(1, 1, 1), rank=0, world=1)
    mask, w = dd.owned_mask(dc)
    assert bool(mask.all())
    out = dd.evaluate(lambda x, t, nloc, bounds: m.eval_local(x, t, nloc, bounds), w.contiguous(), dt)
    torch.cuda.synchronize()
    assert out["nall"] > 2 * len(coord) or name != "W192"
    assert abs(out["energy"].item() - per["energy"].item()) <= 1e-10 * abs(per["energy"].item())
    assert (out["force"] - per["force"]).abs().max().item() <= 2e-9
    assert (out["atom_energy"] - per["atom_energy"]).abs().max().item() <= 1e-10 * per["atom_energy"].abs().max().item()
    assert (out["virial"] - per["virial"]).abs().max().item() <= 1e-10 * max(1.0, per["virial"].abs().max().item())


def test_exchange_kernels_against_numpy():
    """dpb_dd_pack / dpb_dd_unpack / dpb_dd_add_forces (csrc/dd.cu) against the selection written in numpy: same rows
    (as sets: the order inside a message is arbitrary), shifts applied by the sender, counts beyond the capacity reported
    and nothing written past it, forces added at the packed indices."""
    from paper_2004_11658_b200 import binding
    torch = _torch()
    rng = np.random.default_rng(12)
    n = 5000
    x = rng.uniform(0.0, 20.0, size=(n, 3))
    t = rng.integers(0, 3, size=n).astype(np.int32)
    dx, dt = torch.tensor(x, device="cuda"), torch.tensor(t, device="cuda")
    for dim, (cm, cp, sm, sp) in enumerate([(4.0, 16.0, 20.0, -20.0), (3.0, 17.5, 0.0, 0.0), (12.0, 9.0, 20.0, 0.0)]):
        want_m, want_p = np.nonzero(x[:, dim] < cm)[0], np.nonzero(x[:, dim] >= cp)[0]
        cap = n
        pm = torch.full((cap, 4), -7.0, dtype=torch.float64, device="cuda")
        pp = torch.full((cap, 4), -7.0, dtype=torch.float64, device="cuda")
        im = torch.full((cap,), -1, dtype=torch.int32, device="cuda")
        ip = torch.full((cap,), -1, dtype=torch.int32, device="cuda")
        cnt = torch.zeros(2, dtype=torch.int32, device="cuda")
        binding.dd_pack(dx, dt, n, dim, cm, cp, sm, sp, pm, im, pp, ip, cnt)
        km, kp = cnt.tolist()
        assert (km, kp) == (len(want_m), len(want_p))
        for pack, idx, k, want, shift in ((pm, im, km, want_m, sm), (pp, ip, kp, want_p, sp)):
            got_idx = idx[:k].cpu().numpy()
            assert np.array_equal(np.sort(got_idx), want)
            rows = pack[:k].cpu().numpy()
            exp = x[got_idx].copy()
            exp[:, dim] += shift
            assert np.array_equal(rows[:, :3], exp) and np.array_equal(rows[:, 3], t[got_idx].astype(np.float64))
            assert (pack[k:] == -7.0).all() and (idx[k:] == -1).all()
            # unpack and fold forces back
            xo = torch.zeros((k, 3), dtype=torch.float64, device="cuda")
            to = torch.zeros(k, dtype=torch.int32, device="cuda")
            binding.dd_unpack(pack, k, xo, to)
            assert np.array_equal(xo.cpu().numpy(), exp) and np.array_equal(to.cpu().numpy(), t[got_idx])
            f = torch.tensor(rng.normal(size=(n, 3)), device="cuda")
            f0 = f.cpu().numpy().copy()
            fin = torch.tensor(rng.normal(size=(k, 3)), device="cuda")
            binding.dd_add_forces(idx, fin, k, f)
            f0[got_idx] += fin.cpu().numpy()
            assert np.array_equal(f.cpu().numpy(), f0)
        # capacity too small: counts still exact, nothing written beyond the capacity
        small = 64
        pm2 = torch.full((small + 8, 4), -7.0, dtype=torch.float64, device="cuda")
        pp2 = torch.full((small + 8, 4), -7.0, dtype=torch.float64, device="cuda")
        im2 = torch.full((small + 8,), -1, dtype=torch.int32, device="cuda")
        ip2 = torch.full((small + 8,), -1, dtype=torch.int32, device="cuda")
        binding.dd_pack(dx, dt, n, dim, cm, cp, sm, sp, pm2[:small], im2, pp2[:small], ip2, cnt)
        assert cnt.tolist() == [len(want_m), len(want_p)] and len(want_m) > small
        assert (pm2[small:] == -7.0).all() and (im2[small:] == -1).all() and (ip2[small:] == -1).all()
    # empty input
    binding.dd_pack(dx, dt, 0, 0, 1.0, 2.0, 0.0, 0.0, pm, im, pp, ip, cnt)
    assert cnt.tolist() == [0, 0]


def test_triclinic_cell_through_explicit_images():
    """dpb_eval_cell through the C ABI (cell.py only marshals): (1) a genuinely triclinic cell, thinner than 2 r_c
    along c, against the oracle's dpo_eval_local on images built by brute force (tests/test_oracle_local.py);
    (2) W192 described by the sheared cell (a1, a2 + a1, a3 + a2 - a1) against dpb_eval on the orthorhombic box."""
    import paper_2004_11658_b200 as pk
    from paper_2004_11658_b200.cell import eval_cell
    from oracle import Oracle
    from test_oracle_local import _brute_images
    torch = _torch()
    spec, emb, fit = small_model(ntypes=2, s1=8, m_axis=4, fit_width=16, sel=(40, 60), rcut=4.0, rcut_smth=1.0, seed=5,
                                 fit_scale=0.05)
    cell = np.array([[9.0, 0.0, 0.0], [2.5, 8.0, 0.0], [1.0, -1.5, 3.6]])
    rng = np.random.default_rng(8)
    x = rng.uniform(0, 1, size=(40, 3)) @ cell
    t = rng.integers(0, 2, size=40).astype(np.int32)
    orc = Oracle.from_spec(spec, emb, fit)
    xi, own = _brute_images(x, cell, spec.rcut)
    ref = orc.eval_local(xi, t[own], 40, want_nlist=False)
    fref = np.zeros((40, 3))
    np.add.at(fref, own, ref["force"])
    m = pk.DPModel.from_spec(spec, emb, fit)
    got = eval_cell(m, torch.tensor(x, device="cuda"), torch.tensor(t, device="cuda"), cell)
    torch.cuda.synchronize()
    assert abs(got["energy"].item() - ref["energy"]) <= 1e-10 * abs(ref["energy"])
    assert np.abs(got["atom_energy"].cpu().numpy() - ref["atom_energy"]).max() <= 1e-10 * np.abs(ref["atom_energy"]).max()
    assert np.abs(got["force"].cpu().numpy() - fref).max() <= 1e-9
    assert np.abs(got["virial"].cpu().numpy() - ref["virial"]).max() <= 1e-10 * max(1.0, np.abs(ref["virial"]).max())
    m.close()
    # (2)
    spec = MODELS["W192"]
    coord, types, box = gen.make_system("W192")
    emb, fit = gen.make_weights(spec)
    fit = gen.condition_fit_w0(spec, fit)
    m = pk.DPModel.from_spec(spec, emb, fit)
    dc, dt = torch.tensor(coord, device="cuda"), torch.tensor(types, device="cuda")
    per = m.eval(dc, dt, box)
    a = np.asarray(box).reshape(3, 3)
    got = eval_cell(m, dc, dt, np.array([a[0], a[1] + a[0], a[2] + a[1] - a[0]]))
    torch.cuda.synchronize()
    assert abs(got["energy"].item() - per["energy"].item()) <= 1e-10 * abs(per["energy"].item())
    assert (got["force"] - per["force"]).abs().max().item() <= 2e-9
    assert (got["virial"] - per["virial"]).abs().max().item() <= 1e-10 * max(1.0, per["virial"].abs().max().item())
    # (3) the deterministic reduction in a general cell (image rows and the fold are in a fixed order too): bitwise
    # reproducible, same parity, and the per-atom virial [N][9] against the oracle's dpo_atom_virial on the box
    from oracle import Oracle as _O
    av_ref = _O.from_spec(spec, emb, fit).atom_virial(coord, types, box)
    m.set_deterministic(True)
    av = torch.zeros((len(coord), 9), dtype=torch.float64, device="cuda")
    m.set_atom_virial(av)
    sheared = np.array([a[0], a[1] + a[0], a[2] + a[1] - a[0]])
    d1 = eval_cell(m, dc, dt, sheared)
    d1 = {k: v.clone() for k, v in d1.items() if hasattr(v, "clone")}
    d2 = eval_cell(m, dc, dt, sheared)
    torch.cuda.synchronize()
    for k in ("energy", "atom_energy", "force", "virial"):
        assert torch.equal(d1[k], d2[k]), k
    assert (d1["force"] - per["force"]).abs().max().item() <= 2e-9
    assert np.abs(av.cpu().numpy().reshape(-1, 3, 3) - av_ref).max() <= 1e-10 * max(1.0, np.abs(av_ref).max())
    m.set_atom_virial(None)
    m.set_deterministic(False)


def test_subregion_in_several_chunks():
    """dpb_eval_local with a chunk smaller than the number of local atoms (the centres are processed in several chunks,
    the ghosts in none): same result as in one chunk, and parity with the oracle."""
    import paper_2004_11658_b200 as pk
    from oracle import Oracle
    spec = MODELS["W192"]
    coord, types, box = gen.make_system("W192")
    emb, fit = gen.make_weights(spec)
    fit = gen.condition_fit_w0(spec, fit)
    orc = Oracle.from_spec(spec, emb, fit)
    lo, hi = next(iter(bricks(box, (2, 1, 1))))
    loc, own, x, t, bounds = _domain(coord, types, box, lo, hi, spec.rcut)
    ref = orc.eval_local(x, t, len(loc))
    for precision in (0, 1):
        m = pk.DPModel.from_spec(spec, emb, fit, precision=precision)
        m.set_chunk(37)
        got = _gpu_local(m, x, t, len(loc), bounds)
        assert got["info"].n_chunks == (len(loc) + 36) // 37 and got["info"].n_chunks > 2
        _check(ref, got, precision)
        m.close()
