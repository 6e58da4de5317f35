"""GPU parity tests: the CUDA path (through the C ABI, via the thin binding) against the CPU oracle on the same
seeded inputs.  Bars (BASELINE.json north_star): nlist bit-exact including order and padding; fp64: relative error
<= 1e-10 on E, absolute error <= 1e-9 eV/A on F.  We also bound E_i, the virial, T and dT.

All kernel generations are checked: variant 0 (plain unfused kernels), variant 1 (fused DMMA kernels) and variant 2
(the paper's padded-dense, unfused GEMM pipeline as a strawman)."""
import numpy as np
import pytest

import gen
from gen.weights import MODELS, ModelSpec

from conftest import small_model, random_box

pytestmark = pytest.mark.gpu

E_REL = 1e-10
F_ABS = 1e-9


def _torch():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device (the library has no CPU fallback)")
    return torch


def _models(spec, emb, fit, variant):
    from oracle import Oracle
    from paper_2004_11658_b200 import DPModel
    m = DPModel.from_spec(spec, emb, fit)
    m.set_variant(variant)
    return Oracle.from_spec(spec, emb, fit), m


def _gpu_eval(m, coord, types, box, debug=False, spec=None):
    torch = _torch()
    dc = torch.tensor(coord, device="cuda")
    dt = torch.tensor(types, device="cuda")
    dbg = None
    if debug:
        n = coord.shape[0]
        T = torch.zeros((n, spec.m, 4), dtype=torch.float64, device="cuda")
        dT = torch.zeros_like(T)
        m.set_debug_buffers(T, None, dT)
        dbg = (T, dT)
    out = m.eval(dc, dt, box, want_nlist=True, want_info=True)
    torch.cuda.synchronize()
    res = {k: (v.cpu().numpy() if hasattr(v, "cpu") else v) for k, v in out.items()}
    if debug:
        res["T"], res["dT"] = dbg[0].cpu().numpy(), dbg[1].cpu().numpy()
        m.set_debug_buffers(None, None, None)
    return res


def _check_full(ref, got, n_overflow=0):
    assert got["nlist"].dtype == np.int32
    assert np.array_equal(got["nlist"], ref["nlist"]), "nlist must be bit-exact (order and padding)"
    assert got["info"].n_overflow == n_overflow
    e_ref = ref["energy"]
    assert abs(e_ref) >= 1e-3 * np.abs(ref["atom_energy"]).sum()          # reading R20: E is not a cancellation
    assert abs(got["energy"][0] - e_ref) <= E_REL * abs(e_ref)
    assert np.abs(got["atom_energy"] - ref["atom_energy"]).max() <= E_REL * np.abs(ref["atom_energy"]).max()
    assert np.abs(got["force"] - ref["force"]).max() <= F_ABS
    assert np.abs(got["virial"] - ref["virial"]).max() <= 1e-10 * max(1.0, np.abs(ref["virial"]).max())


@pytest.mark.parametrize("variant", [0, 1, 2])
@pytest.mark.parametrize("conditioned", [False, True])
def test_water192_full_parity(variant, conditioned):
    """BASELINE config 0 (W192), literal and conditioned weight sets: every output element against the oracle."""
    spec = MODELS["W192"]
    coord, types, box = gen.make_system("W192")
    emb, fit = gen.make_weights(spec)
    if conditioned:
        fit = gen.condition_fit_w0(spec, fit)
    orc, m = _models(spec, emb, fit, variant)
    ref = orc.eval(coord, types, box)
    got = _gpu_eval(m, coord, types, box, debug=True, spec=spec)
    _check_full(ref, got)
    ar = orc.atom_rows(coord, types, box, None, ref["nlist"], want_T=True)
    assert np.abs(got["T"] - ar["T"]).max() <= 1e-12 * np.abs(ar["T"]).max()
    assert np.abs(got["dT"] - ar["dT"]).max() <= 1e-11 * np.abs(ar["dT"]).max()
    assert got["info"].n_real_pairs == int((ref["nlist"] >= 0).sum())
    m.close()


@pytest.mark.parametrize("variant", [0, 1, 2])
def test_copper_small_full_parity(variant):
    """Copper model (sel 512, 32-64-128) on a 6x6x6-cell FCC box (864 atoms, several row tiles + ragged tail)."""
    spec = MODELS["Cu32k"]
    coord, types, box = gen.copper_box(6, 0.05, seed=gen.SEED_BASE + 2)
    emb, fit = gen.make_weights(spec)
    fit = gen.condition_fit_w0(spec, fit)
    orc, m = _models(spec, emb, fit, variant)
    ref = orc.eval(coord, types, box)
    got = _gpu_eval(m, coord, types, box)
    _check_full(ref, got)
    assert got["info"].max_nei[0] == int((ref["nlist"] >= 0).sum(1).max())
    m.close()


@pytest.mark.parametrize("variant", [0, 1, 2])
@pytest.mark.parametrize("chunk", [1, 7, 100000])
def test_chunking_does_not_change_results(variant, chunk):
    """Atom chunking (the memory bound for the 864k-atom config) must give the same result for any chunk size,
    including chunks that straddle a species boundary."""
    spec = MODELS["W192"]
    coord, types, box = gen.make_system("W192")
    emb, fit = gen.make_weights(spec)
    fit = gen.condition_fit_w0(spec, fit)
    orc, m = _models(spec, emb, fit, variant)
    m.set_chunk(chunk)
    ref = orc.eval(coord, types, box)
    got = _gpu_eval(m, coord, types, box)
    _check_full(ref, got)
    m.close()


@pytest.mark.parametrize("variant", [0, 1, 2])
def test_tiny_model_three_types_random_box(variant):
    """A small 3-species model with odd widths (s1 = 5, M^< = 3, width 9) on a random box with unsorted types:
    exercises padding of every tile dimension and ntypes^2 = 9 embedding nets (Remark 1)."""
    spec, emb, fit = small_model(ntypes=3, s1=5, m_axis=3, fit_width=9, sel=(7, 12, 9), rcut=3.5, rcut_smth=0.8,
                                 seed=11, fit_scale=0.02)
    coord, types, box = random_box(150, 9.0, 3, seed=5, min_dist=0.9)
    orc, m = _models(spec, emb, fit, variant)
    ref = orc.eval(coord, types, box)
    got = _gpu_eval(m, coord, types, box)
    assert np.array_equal(got["nlist"], ref["nlist"])
    assert abs(got["energy"][0] - ref["energy"]) <= E_REL * abs(ref["energy"])
    assert np.abs(got["force"] - ref["force"]).max() <= F_ABS
    assert np.abs(got["virial"] - ref["virial"]).max() <= 1e-10 * max(1.0, np.abs(ref["virial"]).max())
    m.close()


@pytest.mark.parametrize("variant", [0, 1, 2])
def test_neighbour_overflow_keeps_nearest(variant):
    """Reading R8: more neighbours than sel[t] -> the nearest sel[t] are kept and the drops are counted."""
    spec, emb, fit = small_model(ntypes=2, s1=4, m_axis=3, fit_width=8, sel=(3, 4), rcut=4.0, rcut_smth=1.0, seed=3)
    coord, types, box = random_box(120, 10.0, 2, seed=9, min_dist=0.9)
    orc, m = _models(spec, emb, fit, variant)
    nl_ref, ovf_ref = orc.build_nlist(coord, types, box)
    assert ovf_ref > 0
    ref = orc.eval(coord, types, box)
    got = _gpu_eval(m, coord, types, box)
    assert np.array_equal(got["nlist"], nl_ref)
    assert got["info"].n_overflow == ovf_ref
    assert abs(got["energy"][0] - ref["energy"]) <= E_REL * abs(ref["energy"])
    assert np.abs(got["force"] - ref["force"]).max() <= F_ABS
    m.close()


def test_unwrapped_coordinates_and_exact_ties():
    """Raw coordinates outside [0, L) are allowed; a simple-cubic lattice with exactly representable coordinates
    gives exact distance ties, broken by atom index."""
    torch = _torch()
    n = 6
    g = np.stack(np.meshgrid(*[np.arange(n)] * 3, indexing="ij"), -1).reshape(-1, 3).astype(np.float64) * 2.0
    rng = np.random.default_rng(3)
    g_shift = g + 12.0 * rng.integers(-2, 3, size=g.shape)        # whole box vectors: same bits after min-image
    types = np.zeros(len(g), dtype=np.int32)
    box = np.diag([2.0 * n] * 3).reshape(9)
    spec = ModelSpec("sc", 1, 4.5, 1.0, (64,), 4, 2, 8, 0)
    emb, fit = gen.make_weights(spec, seed=1)
    orc, m = _models(spec, emb, fit, 0)
    for c in (g, g_shift):
        nl_ref, _ = orc.build_nlist(c, types, box)
        nl, ovf = m.build_nlist(torch.tensor(c, device="cuda"), torch.tensor(types, device="cuda"), box)
        assert np.array_equal(nl.cpu().numpy(), nl_ref)
    m.close()


def test_empty_and_isolated_inputs():
    """N = 0 is legal; an isolated atom has D = 0, E_i = N(0), F = 0 (SURVEY.md §8(c) pins)."""
    torch = _torch()
    spec, emb, fit = small_model()
    orc, m = _models(spec, emb, fit, 1)
    box = np.diag([20.0] * 3).reshape(9)
    out = m.eval(torch.zeros((0, 3), dtype=torch.float64, device="cuda"),
                 torch.zeros((0,), dtype=torch.int32, device="cuda"), box, want_info=True)
    torch.cuda.synchronize()
    assert out["energy"].item() == 0.0
    coord = np.array([[1.0, 2.0, 3.0], [11.0, 12.0, 13.0]])
    types = np.array([0, 1], dtype=np.int32)
    ref = orc.eval(coord, types, box)
    got = _gpu_eval(m, coord, types, box)
    assert np.all(got["nlist"] == -1)
    assert np.abs(got["atom_energy"] - ref["atom_energy"]).max() <= 1e-14
    assert np.all(got["force"] == 0.0)
    m.close()


def test_errors_are_reported_not_thrown_from_c():
    from paper_2004_11658_b200 import DPBError
    torch = _torch()
    spec, emb, fit = small_model()
    _, m = _models(spec, emb, fit, 1)
    coord = torch.zeros((4, 3), dtype=torch.float64, device="cuda")
    types = torch.zeros((4,), dtype=torch.int32, device="cuda")
    for setter, bad in ((m.lib.dpb_model_set_stored_activations, 2), (m.lib.dpb_model_set_pair_reuse, 3)):
        assert setter(m._h, bad) == -1 and b"0" in m.lib.dpb_last_error()   # DPB_EINVAL, message names the values
    with pytest.raises(DPBError) as e:
        m.eval(coord, types, np.diag([7.0] * 3).reshape(9))                  # r_c = 4 >= L/2
    assert e.value.status == -2
    skew = np.diag([20.0] * 3); skew[0, 1] = 1.0
    with pytest.raises(DPBError) as e:
        m.eval(coord, types, skew.reshape(9))
    assert e.value.status == -2
    bad = torch.full((4,), 5, dtype=torch.int32, device="cuda")
    with pytest.raises(DPBError) as e:
        m.eval(torch.rand((4, 3), dtype=torch.float64, device="cuda") * 20, bad, np.diag([20.0] * 3).reshape(9),
               want_info=True)
    assert e.value.status == -1
    m.close()


@pytest.mark.parametrize("conditioned", [False, True])
@pytest.mark.parametrize("name", ["W24k", "Cu32k"])
def test_full_size_parity_every_element(name, conditioned):
    """BASELINE configs 1 and 2 at full size, in the launch configuration bench.py times (variant 1, default chunk,
    default pair reuse) and on the weight set it times (literal) as well as the conditioned one: EVERY output element
    against the oracle's whole evaluation — nlist bit-exact on all rows, E, E_i, every force component, the virial
    (Eq. 10; ProdForce / ProdVirial :240), T and dT through the debug buffers on sampled rows.
    The pair reuse and the stored activations are also switched off and on again (one chunk and several); the two kernel
    generations are compared as an extra."""
    from conftest import oracle_full
    torch = _torch()
    spec, emb, fit, coord, types, box, ref = oracle_full(name, conditioned)
    orc, m = _models(spec, emb, fit, 1)
    got = _gpu_eval(m, coord, types, box, debug=True, spec=spec)
    _check_full(ref, got)
    assert got["info"].n_real_pairs == int((ref["nlist"] >= 0).sum())
    rows = np.random.default_rng(1).choice(coord.shape[0], 48, replace=False).astype(np.int64)
    ar = orc.atom_rows(coord, types, box, rows, ref["nlist"][rows], want_T=True)
    assert np.abs(got["T"][rows] - ar["T"]).max() <= 1e-12 * np.abs(ar["T"]).max()
    assert np.abs(got["dT"][rows] - ar["dT"]).max() <= 1e-11 * np.abs(ar["dT"]).max()
    assert abs(got["energy"][0] - got["atom_energy"].sum()) <= 1e-12 * np.abs(got["atom_energy"]).sum()
    for reuse in (0, 2):
        m.set_pair_reuse(reuse)
        _check_full(ref, _gpu_eval(m, coord, types, box))
    # stored activations (default on: the runs above) off, and on again in several chunks — pass 1 then evaluates every
    # row (pair_reuse 1) or shares inside a chunk only (2), pass 2 reads the records of the rows of the lower atom
    m.set_pair_reuse(1)
    m.set_stored_activations(False)
    _check_full(ref, _gpu_eval(m, coord, types, box))
    m.set_stored_activations(True)
    m.set_species_pipeline(False)                              # (default on: every run above, for the water box)
    _check_full(ref, _gpu_eval(m, coord, types, box))
    m.set_species_pipeline(True)
    m.set_chunk(8192)
    for reuse in (1, 2):
        m.set_pair_reuse(reuse)
        got = _gpu_eval(m, coord, types, box)
        assert got["info"].n_chunks >= 3
        _check_full(ref, got)
    m.close()
    if not conditioned:
        m0 = _models(spec, emb, fit, 0)[1]
        _check_full(ref, _gpu_eval(m0, coord, types, box))
        m0.close()


@pytest.mark.parametrize("s1,sel", [(8, (40, 60, 30)), (16, (40, 60, 30)), (8, (5, 7, 4))])
def test_stored_activations_other_net_widths_and_overflow(s1, sel):
    """The stored-activation kernels in their other instantiations (s1 = 8, 16: SP = 2, 4; the BASELINE configs use 7
    and 8) on a 5,400-atom, 3-species box (a chunk of >= 4,096 centres is what switches them on), and with sections so
    short that neighbours are dropped: the pair reuse then switches itself off on the device while pass 2 still reads the
    records.  Every output element against the oracle, stored activations on and off."""
    spec, emb, fit = small_model(ntypes=3, s1=s1, m_axis=4, fit_width=16, sel=sel, rcut=4.0, rcut_smth=1.0, seed=12,
                                 fit_scale=0.05)
    c0, t0, b0 = random_box(200, 10.0, 3, seed=31, min_dist=1.1)
    shifts = np.array([[i, j, k] for i in range(3) for j in range(3) for k in range(3)], dtype=np.float64) * 10.0
    coord = (c0[None, :, :] + shifts[:, None, :]).reshape(-1, 3)
    coord = coord + np.random.default_rng(5).normal(0.0, 0.02, size=coord.shape)
    types = np.tile(t0, 27)
    box = np.diag([30.0, 30.0, 30.0]).reshape(-1)
    orc, m = _models(spec, emb, fit, 1)
    ref = orc.eval(coord, types, box)
    _, ovf = orc.build_nlist(coord, types, box)
    assert (ovf > 0) == (sel[0] < 10)
    torch = _torch()
    on = _gpu_eval(m, coord, types, box)
    _check_full(ref, on, n_overflow=ovf)
    free_on = torch.cuda.mem_get_info()[0]
    m.set_stored_activations(False)                            # releases the records: that they existed shows the path ran
    off = _gpu_eval(m, coord, types, box)
    _check_full(ref, off, n_overflow=ovf)
    sp = (s1 + 3) // 4
    records = len(coord) * sum(sel) * 4 * (((sp + 1) & ~1) + 6 * sp) * 8
    assert torch.cuda.mem_get_info()[0] - free_on >= 0.9 * records
    assert np.abs(on["force"] - off["force"]).max() <= 1e-12 * max(1.0, np.abs(off["force"]).max())
    m.close()


def test_exactly_4096_atoms_where_the_small_and_the_large_paths_meet():
    """4,096 atoms, two species: the evaluation is at once a 'small' one (graph replay, folded memsets, energy sum beside
    pass 2) and a 'large' one (whole-atom work items, stored activations, species pipeline).  Every output element against
    the oracle, eagerly and replayed from the graph."""
    torch = _torch()
    spec, emb, fit = small_model(ntypes=2, s1=8, m_axis=4, fit_width=16, sel=(40, 60), rcut=4.0, rcut_smth=1.0, seed=23,
                                 fit_scale=0.05)
    c0, t0, b0 = random_box(256, 11.0, 2, seed=41, min_dist=1.1)
    shifts = np.array([[i, j, k] for i in range(2) for j in range(2) for k in range(4)], dtype=np.float64) * 11.0
    coord = (c0[None, :, :] + shifts[:, None, :]).reshape(-1, 3)
    coord = coord + np.random.default_rng(6).normal(0.0, 0.02, size=coord.shape)
    types = np.tile(t0, 16)
    box = np.diag([22.0, 22.0, 44.0]).reshape(-1)
    assert len(coord) == 4096
    orc, m = _models(spec, emb, fit, 1)
    ref = orc.eval(coord, types, box)
    _check_full(ref, _gpu_eval(m, coord, types, box))
    dc, dt = torch.tensor(coord, device="cuda"), torch.tensor(types.astype(np.int32), device="cuda")
    out = None
    for _ in range(3):                                         # eager, captured, replayed
        out = m.eval(dc, dt, box, out=out)
        torch.cuda.synchronize()
        assert abs(out["energy"].item() - ref["energy"]) <= E_REL * abs(ref["energy"])
        assert np.abs(out["force"].cpu().numpy() - ref["force"]).max() <= F_ABS
    m.close()


@pytest.mark.parametrize("fit_width", [48, 96, 144])
def test_small_system_cluster_kernel_other_widths(fit_width):
    """The cluster kernel of the small-system fitting chain (k_fit_mid_cluster: widths that are multiples of 48, clusters of
    w / 48 CTAs; BASELINE configs[0] runs it with 5) with clusters of 1, 2 and 3 CTAs, on a 2-species box whose species
    have ragged last tiles (70 + 50 atoms: tiles of 16 rows), every output element against the oracle."""
    spec, emb, fit = small_model(ntypes=2, s1=8, m_axis=4, fit_width=fit_width, sel=(30, 40), rcut=4.0, rcut_smth=1.0,
                                 seed=17, fit_scale=0.05)
    coord, types, box = random_box(120, 11.0, 2, seed=4, min_dist=1.1)
    types[:70] = 0; types[70:] = 1
    orc, m = _models(spec, emb, fit, 1)
    ref = orc.eval(coord, types, box)
    got = _gpu_eval(m, coord, types, box)
    _check_full(ref, got)
    m.close()


def test_eval_host_matches_device_entry():
    """dpb_eval_host (host buffers, copies inside) returns the same numbers as dpb_eval."""
    torch = _torch()
    spec = MODELS["W192"]
    coord, types, box = gen.make_system("W192")
    emb, fit = gen.make_weights(spec)
    _, m = _models(spec, emb, fit, 1)
    dev = _gpu_eval(m, coord, types, box)
    host = m.eval_host(coord, types, box, want_nlist=True)
    assert np.array_equal(host["nlist"], dev["nlist"])
    assert np.abs(host["force"] - dev["force"]).max() <= 1e-12
    assert abs(host["energy"][0] - dev["energy"][0]) <= 1e-12 * abs(dev["energy"][0])
    m.close()


@pytest.mark.parametrize("conditioned,chunk", [(False, 0), (True, 32768)])
def test_config5_copper_864k_sampled(conditioned, chunk):
    """BASELINE configs[4]: 864,000-atom copper box, in the launch configuration bench.py times (automatic chunk: one chunk
    on an otherwise empty B200) and as 27 chunks of 32,768 atoms; too large for a whole oracle evaluation
    inside the test budget.  Against the oracle, element by element, on sampled atoms — 16 random ones plus the two
    atoms on either side of four chunk boundaries (sorted order through dpb_debug_sorted_order): nlist rows bit-exact,
    E_i, and the FORCE, assembled from the oracle's per-row pieces F_i = sum_k f_ik - sum_{j: i in L(j)} f_{j,slot(i)}
    over the atom and all of its neighbours (conftest.oracle_forces_of).  Whole-box properties: sum F = 0, symmetric
    virial, E = sum E_i.  The box is not a replica of config 2 (independent jitter), so no extensivity check."""
    from conftest import oracle_forces_of
    torch = _torch()
    spec = MODELS["Cu864k"]
    coord, types, box = gen.make_system("Cu864k")
    emb, fit = gen.make_weights(spec)
    if conditioned:
        fit = gen.condition_fit_w0(spec, fit)
    orc, m = _models(spec, emb, fit, 1)
    if chunk:
        m.set_chunk(chunk)
    dc = torch.tensor(coord, device="cuda")
    dt = torch.tensor(types, device="cuda")
    out = m.eval(dc, dt, box, want_nlist=True, want_info=True)
    torch.cuda.synchronize()
    info = out["info"]
    assert info.n_overflow == 0 and (info.n_chunks == 27 if chunk else info.n_chunks >= 1)
    order = m.sorted_order(coord.shape[0]).cpu().numpy().astype(np.int64)
    assert np.array_equal(np.sort(order), np.arange(coord.shape[0]))
    edge = [order[c * 32768 + d] for c in (1, 9, 17, 26) for d in (-1, 0)]    # chunk boundaries of the 27-chunk run
    atoms = np.unique(np.concatenate([np.random.default_rng(2).choice(coord.shape[0], 16, replace=False), edge]))
    F_ref, E_ref, nl_ref = oracle_forces_of(orc, coord, types, box, atoms)
    sel = torch.tensor(atoms, device="cuda")
    assert np.array_equal(out["nlist"][sel].cpu().numpy(), nl_ref)
    ei = out["atom_energy"].cpu().numpy()
    assert np.abs(ei[atoms] - E_ref).max() <= E_REL * np.abs(E_ref).max()
    f = out["force"].cpu().numpy()
    assert np.abs(f[atoms] - F_ref).max() <= F_ABS
    assert np.abs(f.sum(0)).max() <= 1e-9
    v = out["virial"].cpu().numpy()
    assert np.abs(v - v.T).max() <= 1e-9 * np.abs(v).max()
    assert abs(out["energy"].item() - ei.sum()) <= 1e-11 * np.abs(ei).sum()
    m.close()


def test_replication_extensivity_gpu():
    """A 2x2x2 periodic replication gives exactly 8 E and replicated forces (PBC + cell list + chunking), here with
    a chunk size that does not divide the atom count."""
    torch = _torch()
    spec = MODELS["W192"]
    coord, types, box = gen.make_system("W192")
    emb, fit = gen.make_weights(spec)
    fit = gen.condition_fit_w0(spec, fit)
    _, m = _models(spec, emb, fit, 1)
    small = _gpu_eval(m, coord, types, box)
    big_c, big_t, big_b = gen.replicate(coord, types, box, 2)
    m.set_chunk(500)
    big = _gpu_eval(m, big_c, big_t, big_b)
    assert abs(big["energy"][0] - 8 * small["energy"][0]) <= 1e-11 * abs(8 * small["energy"][0])
    assert np.abs(big["force"].reshape(8, -1, 3) - small["force"][None]).max() <= 1e-10
    assert np.abs(big["virial"] - 8 * small["virial"]).max() <= 1e-10 * np.abs(8 * small["virial"]).max()
    m.close()


@pytest.mark.parametrize("chunk", [100000, 50])
def test_deterministic_reduction(chunk):
    """SURVEY.md §7 hard part 6: forces and virial gathered in a fixed order (no atomics).  Two evaluations agree bit for
    bit, the result matches the oracle to the fp64 bar and the atomics mode to rounding; also with chunks that cut the
    species ranges (the gather needs every atom's row)."""
    torch = _torch()
    spec = MODELS["W192"]
    coord, types, box = gen.make_system("W192")
    emb, fit = gen.make_weights(spec)
    fit = gen.condition_fit_w0(spec, fit)
    orc, m = _models(spec, emb, fit, 1)
    m.set_chunk(chunk)
    ref = orc.eval(coord, types, box)
    atom = _gpu_eval(m, coord, types, box)
    m.set_deterministic(True)
    d1 = _gpu_eval(m, coord, types, box)
    d2 = _gpu_eval(m, coord, types, box)
    _check_full(ref, d1)
    assert np.array_equal(d1["force"], d2["force"]) and np.array_equal(d1["virial"], d2["virial"])
    assert d1["energy"][0] == d2["energy"][0]
    assert np.abs(d1["force"] - atom["force"]).max() <= 1e-12
    assert np.abs(d1["virial"] - atom["virial"]).max() <= 1e-12 * np.abs(atom["virial"]).max()
    m.close()


def test_deterministic_reduction_full_size_is_bitwise_reproducible():
    """W24k: the atomics mode differs between two runs in the last bits of some forces; the deterministic mode does not."""
    torch = _torch()
    spec = MODELS["W24k"]
    coord, types, box = gen.make_system("W24k")
    emb, fit = gen.make_weights(spec)
    _, m = _models(spec, emb, fit, 1)
    a1 = _gpu_eval(m, coord, types, box)
    m.set_deterministic(True)
    d1 = _gpu_eval(m, coord, types, box)
    d2 = _gpu_eval(m, coord, types, box)
    assert np.array_equal(d1["force"], d2["force"]) and np.array_equal(d1["virial"], d2["virial"])
    assert np.abs(d1["force"] - a1["force"]).max() <= 1e-11
    assert np.abs(d1["force"].sum(0)).max() <= 1e-9
    m.close()


def test_deterministic_mode_is_refused_where_it_is_not_built():
    from paper_2004_11658_b200 import DPBError
    torch = _torch()
    spec, emb, fit = small_model()
    _, m = _models(spec, emb, fit, 0)
    m.set_deterministic(True)
    coord, types, box = random_box(40, 10.0, 2, seed=2, min_dist=1.0)
    with pytest.raises(DPBError) as e:
        m.eval(torch.tensor(coord, device="cuda"), torch.tensor(types, device="cuda"), box)
    assert e.value.status == -6
    m.close()


def test_atom_virial_against_the_oracle():
    """Per-atom virial (centre-atom split, include/dpb.h) from the deterministic gather: every
    component of every atom against dpo_atom_virial on W192 and on a 3-species box; its sum equals the virial output;
    without the deterministic reduction the request is refused."""
    torch = _torch()
    from paper_2004_11658_b200 import DPBError
    cases = []
    spec = MODELS["W192"]
    coord, types, box = gen.make_system("W192")
    emb, fit = gen.make_weights(spec)
    cases.append((spec, emb, gen.condition_fit_w0(spec, fit), coord, types, box))
    spec3, emb3, fit3 = small_model(ntypes=3, s1=5, m_axis=3, fit_width=9, sel=(24, 30, 30), rcut=3.5, rcut_smth=0.8, seed=11)
    c3, t3, b3 = random_box(150, 9.0, 3, seed=5, min_dist=0.9)
    cases.append((spec3, emb3, fit3, c3, t3, b3))
    for spec, emb, fit, coord, types, box in cases:
        orc, m = _models(spec, emb, fit, 1)
        ref = orc.atom_virial(coord, types, box)
        dc, dt = torch.tensor(coord, device="cuda"), torch.tensor(types, device="cuda")
        av = torch.full((len(coord), 9), float("nan"), dtype=torch.float64, device="cuda")
        m.set_atom_virial(av)
        with pytest.raises(DPBError):
            m.eval(dc, dt, box)
        m.set_deterministic(True)
        out = m.eval(dc, dt, box, want_info=True)
        torch.cuda.synchronize()
        assert out["info"].n_overflow == 0
        got = av.cpu().numpy().reshape(-1, 3, 3)
        assert np.abs(got - ref).max() <= 1e-10 * max(1.0, np.abs(ref).max())
        assert np.abs(got.sum(axis=0) - out["virial"].cpu().numpy()).max() <= 1e-10 * max(1.0, np.abs(ref.sum(axis=0)).max())
        m.set_atom_virial(None)
        m.set_deterministic(False)
        m.eval(dc, dt, box)
        m.close()


@pytest.mark.parametrize("name,chunk", [("W192", 100000), ("W192", 50), ("Cu-small", 100000)])
def test_pair_reuse_matches_oracle_and_the_plain_pass(name, chunk):
    """Same-species pair reuse in pass 1 (dpb_model_set_pair_reuse, on by default): T (Eq. 4's G^T R~, checked through the
    debug buffer), E, F and the virial against the oracle with the reuse on, and against the pass without it; with
    chunks the pairs that straddle a chunk boundary are evaluated in both directions."""
    if name == "W192":
        spec = MODELS["W192"]
        coord, types, box = gen.make_system("W192")
    else:
        spec = MODELS["Cu32k"]
        coord, types, box = gen.copper_box(6, 0.05, seed=gen.SEED_BASE + 2)
    emb, fit = gen.make_weights(spec)
    fit = gen.condition_fit_w0(spec, fit)
    orc, m = _models(spec, emb, fit, 1)
    m.set_chunk(chunk)
    ref = orc.eval(coord, types, box)
    res = {}
    for on in (True, False):
        m.set_pair_reuse(2 if on else 0)                # 2: also when the evaluation runs in several chunks
        res[on] = _gpu_eval(m, coord, types, box, debug=True, spec=spec)
        _check_full(ref, res[on])
    scale = np.abs(res[False]["T"]).max()
    assert np.abs(res[True]["T"] - res[False]["T"]).max() <= 1e-13 * scale
    assert np.abs(res[True]["force"] - res[False]["force"]).max() <= 1e-11
    m.close()


def test_staging_capacity_overflow_is_reported_and_touches_no_unwritten_slot():
    """More in-range candidates than the staging capacity max(256, 2 Nm) (a mis-scaled, far too dense input): the call
    with info reports DPB_ECAP; the overflowing rows are written empty (all -1), so the passes enqueued behind the
    neighbour kernel read no stale slot — the call without info runs through, outputs are finite, dpb_model_status
    then reports the error, and the model still evaluates a sane input correctly afterwards."""
    from paper_2004_11658_b200 import DPBError
    torch = _torch()
    spec, emb, fit = small_model(ntypes=1, s1=4, m_axis=3, fit_width=8, sel=(20,), rcut=4.0, rcut_smth=1.0, seed=5)
    orc, m = _models(spec, emb, fit, 1)
    rng = np.random.default_rng(12)
    n = 2000                                             # 2000 atoms in a 9 A box: ~730 atoms inside r_c = 4 > cap = 256
    coord = rng.uniform(0, 9.0, (n, 3))
    types = np.zeros(n, dtype=np.int32)
    box = np.diag([9.0] * 3).reshape(9)
    dc, dt = torch.tensor(coord, device="cuda"), torch.tensor(types, device="cuda")
    with pytest.raises(DPBError) as e:
        m.eval(dc, dt, box, want_info=True)
    assert e.value.status == -5
    out = m.eval(dc, dt, box, want_nlist=True)           # no info: DPB_OK now, the error is deferred
    torch.cuda.synchronize()
    assert bool((out["nlist"] == -1).all())
    assert bool(torch.isfinite(out["force"]).all()) and bool(torch.isfinite(out["atom_energy"]).all())
    with pytest.raises(DPBError) as e:
        m.status()
    assert e.value.status == -5
    coord2, types2, box2 = random_box(60, 10.0, 1, seed=2, min_dist=1.0)
    ref = orc.eval(coord2, types2, box2)
    got = _gpu_eval(m, coord2, types2, box2)
    assert np.array_equal(got["nlist"], ref["nlist"])
    assert np.abs(got["force"] - ref["force"]).max() <= F_ABS
    m.status()
    m.close()


def test_cuda_graph_replay_matches_the_oracle():
    """dpb_model_set_graph (default: evaluations of at most 4096 atoms): the first call with an argument set runs eagerly,
    the second is captured, later ones replay the graph.  Calls 1-4 on two alternating coordinate buffers (W192, fresh
    perturbations written INTO the same device buffers between calls) are each compared with the oracle; the kernel
    counter advances by the same amount per call whether eager or replayed; mode 0 gives the same numbers."""
    torch = _torch()
    spec = MODELS["W192"]
    coord, types, box = gen.make_system("W192")
    emb, fit = gen.make_weights(spec)
    fit = gen.condition_fit_w0(spec, fit)
    orc, m = _models(spec, emb, fit, 1)
    bufs = [torch.empty((192, 3), dtype=torch.float64, device="cuda") for _ in range(2)]
    dt = torch.tensor(types, device="cuda")
    outs = [None, None]
    per_call = []
    for call in range(8):
        c = gen.perturbed(coord, box, 0.01, 77 + call)
        b = call % 2
        bufs[b].copy_(torch.tensor(c))
        n0 = m.kernel_launches()
        outs[b] = m.eval(bufs[b], dt, box, want_nlist=True, out=outs[b])
        torch.cuda.synchronize()
        per_call.append(m.kernel_launches() - n0)
        ref = orc.eval(c, types, box)
        got = {k: v.cpu().numpy() for k, v in outs[b].items()}
        assert np.array_equal(got["nlist"], ref["nlist"]), call
        assert abs(got["energy"][0] - ref["energy"]) <= E_REL * abs(ref["energy"]), call
        assert np.abs(got["force"] - ref["force"]).max() <= F_ABS, call
        assert np.abs(got["virial"] - ref["virial"]).max() <= 1e-10 * max(1.0, np.abs(ref["virial"]).max()), call
    assert len(set(per_call)) == 1 and per_call[0] > 0, per_call
    m.set_graph(0)
    n0 = m.kernel_launches()
    eager = m.eval(bufs[1], dt, box)
    torch.cuda.synchronize()
    assert m.kernel_launches() - n0 == per_call[0]
    assert np.abs(eager["force"].cpu().numpy() - outs[1]["force"].cpu().numpy()).max() <= 1e-12
    m.close()
