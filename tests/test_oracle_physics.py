"""Whole-model pins for the oracle: F = -grad E by finite differences, sum F = 0, invariances, virial against
strain differences and against sum r (x) F, extensivity, and an independent PyTorch-autograd restatement of
Eq. 1-10 (dense N x N masks, library matmuls, autograd for every derivative).  No CUDA here."""
import numpy as np
import pytest
import torch

import gen
from gen.weights import emb_net_size, fit_net_size
from oracle import Oracle

from conftest import small_model, random_box


# ----------------------------------------------------------------------------- independent autograd model
def _split_emb(p, s1):
    W0, b0 = p[:s1], p[s1:2 * s1]
    q = p[2 * s1:]
    W1, b1 = q[:s1 * 2 * s1].reshape(s1, 2 * s1), q[s1 * 2 * s1: s1 * 2 * s1 + 2 * s1]
    q = q[s1 * 2 * s1 + 2 * s1:]
    W2, b2 = q[:2 * s1 * 4 * s1].reshape(2 * s1, 4 * s1), q[2 * s1 * 4 * s1: 2 * s1 * 4 * s1 + 4 * s1]
    return W0, b0, W1, b1, W2, b2


def autograd_model(spec, emb, fit, coord, types, box, strain=None):
    """E, E_i, F, virial from torch autograd.  Order-free formulation: T_i = sum_j mask_ij g_ij (x) R~_ij, so it
    shares neither the neighbour list nor the backward formulas with the oracle."""
    dt = torch.float64
    x = torch.tensor(coord, dtype=dt, requires_grad=True)
    eps = torch.zeros(3, 3, dtype=dt, requires_grad=True)
    Lvec = torch.tensor([box[0], box[4], box[8]], dtype=dt)
    tt = torch.tensor(types, dtype=torch.long)
    n = x.shape[0]
    # integer image shifts from the unstrained geometry (constants), then strain coordinates and box together
    d0 = x.detach()[None, :, :] - x.detach()[:, None, :]
    shift = torch.round(d0 / Lvec)
    d = (x[None, :, :] - x[:, None, :]) - shift * Lvec            # d[i, j] = r_j - r_i (minimum image)
    d = d + d @ eps.T                                            # homogeneous strain r -> (I + eps) r
    eye = torch.eye(n, dtype=torch.bool)
    r = torch.sqrt((d * d).sum(-1) + eye.to(dt))                 # avoid sqrt(0) on the diagonal
    u = (r - spec.rcut_smth) / (spec.rcut - spec.rcut_smth)
    w = torch.where(r < spec.rcut_smth, torch.ones_like(r),
                    torch.where(r < spec.rcut, u ** 3 * (-6 * u ** 2 + 15 * u - 10) + 1, torch.zeros_like(r)))
    mask = (r <= spec.rcut) & (~eye)
    s = torch.where(mask, w / r, torch.zeros_like(r))
    env = torch.cat([s[..., None], (s / r)[..., None] * d], dim=-1)          # [n, n, 4]
    s1, M, Ma, wd = spec.emb_s1, spec.m, spec.m_axis, spec.fit_width
    embt = torch.tensor(emb, dtype=dt)
    fitt = torch.tensor(fit, dtype=dt)
    T = torch.zeros(n, M, 4, dtype=dt)
    for a in range(spec.ntypes):
        ia = torch.where(tt == a)[0]
        for t in range(spec.ntypes):
            jt = torch.where(tt == t)[0]
            if len(ia) == 0 or len(jt) == 0:
                continue
            W0, b0, W1, b1, W2, b2 = _split_emb(embt[(a * spec.ntypes + t) * emb_net_size(s1):], s1)
            sx = s[ia][:, jt]                                                  # [na, nt]
            h0 = torch.tanh(sx[..., None] * W0 + b0)
            h1 = torch.cat([h0, h0], -1) + torch.tanh(h0 @ W1 + b1)
            g = torch.cat([h1, h1], -1) + torch.tanh(h1 @ W2 + b2)             # [na, nt, M]
            g = g * mask[ia][:, jt][..., None].to(dt)
            T = T.index_add(0, ia, torch.einsum("ijb,ijc->ibc", g, env[ia][:, jt]))
    D = torch.einsum("ibc,iac->iba", T, T[:, :Ma, :]).reshape(n, M * Ma)
    ei = torch.zeros(n, dtype=dt)
    dim = M * Ma
    for a in range(spec.ntypes):
        ia = torch.where(tt == a)[0]
        p = fitt[a * fit_net_size(dim, wd):]
        W0, p = p[:dim * wd].reshape(dim, wd), p[dim * wd:]
        b0, p = p[:wd], p[wd:]
        W1, p = p[:wd * wd].reshape(wd, wd), p[wd * wd:]
        b1, p = p[:wd], p[wd:]
        W2, p = p[:wd * wd].reshape(wd, wd), p[wd * wd:]
        b2, p = p[:wd], p[wd:]
        w3, b3 = p[:wd], p[wd]
        z0 = torch.tanh(D[ia] @ W0 + b0)
        z1 = z0 + torch.tanh(z0 @ W1 + b1)
        z2 = z1 + torch.tanh(z1 @ W2 + b2)
        ei = ei.index_add(0, ia, z2 @ w3 + b3)
    E = ei.sum()
    gx, geps = torch.autograd.grad(E, [x, eps])
    return dict(energy=float(E.detach()), atom_energy=ei.detach().numpy(), force=-gx.numpy(), virial=-geps.numpy())


@pytest.mark.parametrize("which", ["literal", "conditioned"])
def test_oracle_matches_autograd_water192(which, water192, water192_cond):
    cfg = water192 if which == "literal" else water192_cond
    ref = autograd_model(cfg["spec"], cfg["emb"], cfg["fit"], cfg["coord"], cfg["types"], cfg["box"])
    out = cfg["oracle"].eval(cfg["coord"], cfg["types"], cfg["box"])
    assert abs(out["energy"] - ref["energy"]) <= 1e-12 * np.abs(ref["atom_energy"]).sum()
    assert np.allclose(out["atom_energy"], ref["atom_energy"], rtol=0, atol=1e-11)
    frms = np.sqrt((ref["force"] ** 2).mean())
    assert frms > 1e-3
    assert np.abs(out["force"] - ref["force"]).max() <= 1e-11 * max(1.0, frms)
    vref = ref["virial"]
    assert np.abs(out["virial"] - vref).max() <= 1e-11 * np.abs(vref).max()
    assert np.abs(out["virial"].T - vref).max() <= 1e-11 * np.abs(vref).max()    # symmetric


def test_oracle_matches_autograd_small_three_species():
    spec, emb, fit = small_model(ntypes=3, s1=5, m_axis=4, fit_width=10, sel=(30, 30, 30), rcut=3.5)
    coord, types, box = random_box(90, 8.0, 3, seed=21)
    ref = autograd_model(spec, emb, fit, coord, types, box)
    out = Oracle.from_spec(spec, emb, fit).eval(coord, types, box)
    assert abs(out["energy"] - ref["energy"]) <= 1e-12 * np.abs(ref["atom_energy"]).sum()
    assert np.abs(out["force"] - ref["force"]).max() <= 1e-12 * max(1.0, np.abs(ref["force"]).max())
    assert np.abs(out["virial"] - ref["virial"]).max() <= 1e-12 * max(1.0, np.abs(ref["virial"]).max())


# ----------------------------------------------------------------------------- properties of the oracle alone
def test_forces_are_minus_gradient_finite_differences(water192_cond):
    cfg = water192_cond
    o, coord, types, box = cfg["oracle"], cfg["coord"], cfg["types"], cfg["box"]
    base = o.eval(coord, types, box)
    h = 1e-5
    rng = np.random.default_rng(0)
    for i, c in zip(rng.integers(0, 192, 6), rng.integers(0, 3, 6)):
        cp, cm = coord.copy(), coord.copy()
        cp[i, c] += h
        cm[i, c] -= h
        fd = -(o.eval(cp, types, box)["energy"] - o.eval(cm, types, box)["energy"]) / (2 * h)
        assert abs(fd - base["force"][i, c]) < 2e-7 * max(1.0, abs(fd))


def test_sum_of_forces_vanishes(water192, water192_cond):
    for cfg in (water192, water192_cond):
        out = cfg["oracle"].eval(cfg["coord"], cfg["types"], cfg["box"])
        assert np.abs(out["force"].sum(0)).max() < 1e-12 * np.abs(out["force"]).sum()


def test_translation_invariance_across_the_boundary(water192_cond):
    cfg = water192_cond
    o = cfg["oracle"]
    a = o.eval(cfg["coord"], cfg["types"], cfg["box"])
    b = o.eval(cfg["coord"] + np.array([5.3, -17.1, 40.7]), cfg["types"], cfg["box"])   # unwrapped raw coords
    scale = np.abs(a["atom_energy"]).sum()
    assert abs(a["energy"] - b["energy"]) < 1e-12 * scale
    assert np.abs(a["force"] - b["force"]).max() < 1e-11
    assert np.array_equal(a["nlist"], b["nlist"]) or (a["nlist"] != b["nlist"]).mean() < 0.01


def test_same_type_permutation(water192_cond):
    cfg = water192_cond
    o = cfg["oracle"]
    a = o.eval(cfg["coord"], cfg["types"], cfg["box"])
    rng = np.random.default_rng(4)
    perm = np.arange(192)
    for t in (0, 1):
        idx = np.where(cfg["types"] == t)[0]
        perm[idx] = rng.permutation(idx)
    b = o.eval(cfg["coord"][perm], cfg["types"][perm], cfg["box"])
    assert np.array_equal(cfg["types"][perm], cfg["types"])
    assert abs(a["energy"] - b["energy"]) < 1e-12 * np.abs(a["atom_energy"]).sum()
    assert np.abs(a["force"][perm] - b["force"]).max() < 1e-11
    assert np.abs(a["atom_energy"][perm] - b["atom_energy"]).max() < 1e-11


def test_rotation_of_a_cluster(water192_cond):
    """A cluster in a box so large that nothing interacts across the boundary: E invariant, F rotates, and the
    virial equals sum_i r_i (x) F_i."""
    cfg = water192_cond
    o = cfg["oracle"]
    big = np.diag([60.0] * 3).reshape(9)
    x = cfg["coord"][:96] + 20.0                       # 32 molecules, extent ~12.4 A, far from any image
    t = cfg["types"][:96]
    a = o.eval(x, t, big)
    from gen.systems import _random_rotations
    R = _random_rotations(np.random.default_rng(2), 1)[0]
    c0 = x.mean(0)
    xr = (x - c0) @ R.T + c0
    b = o.eval(xr, t, big)
    assert abs(a["energy"] - b["energy"]) < 1e-12 * np.abs(a["atom_energy"]).sum()
    assert np.abs(a["force"] @ R.T - b["force"]).max() < 1e-11
    assert np.abs(R @ a["virial"] @ R.T - b["virial"]).max() < 1e-10
    rf = np.einsum("ia,ib->ab", x, a["force"])
    assert np.abs(rf - a["virial"]).max() < 1e-10 * max(1.0, np.abs(a["virial"]).max())


def test_virial_is_minus_strain_derivative(water192_cond):
    cfg = water192_cond
    o, coord, types, box = cfg["oracle"], cfg["coord"], cfg["types"], cfg["box"]
    vir = o.eval(coord, types, box)["virial"]
    h = 1e-6
    for (a, b) in ((0, 0), (1, 1), (2, 2)):           # diagonal strains keep the box orthorhombic
        e = []
        for sgn in (+1, -1):
            F = np.eye(3)
            F[a, b] += sgn * h
            e.append(o.eval(coord @ F.T, types, (box.reshape(3, 3) @ F.T).reshape(9))["energy"])
        fd = -(e[0] - e[1]) / (2 * h)
        assert abs(fd - vir[a, b]) < 5e-7 * max(1.0, abs(fd))
    assert np.abs(vir - vir.T).max() < 1e-11 * np.abs(vir).max()


def test_extensivity_under_replication(water192_cond):
    """2x2x2 periodic replication: exactly 8 E and replicated forces (strong test of PBC handling)."""
    cfg = water192_cond
    o = cfg["oracle"]
    a = o.eval(cfg["coord"], cfg["types"], cfg["box"])
    big, tb, bb = gen.replicate(cfg["coord"], cfg["types"], cfg["box"], 2)
    b = o.eval(big, tb, bb, cells=True)
    assert abs(b["energy"] - 8 * a["energy"]) < 1e-11 * 8 * np.abs(a["atom_energy"]).sum()
    assert np.abs(b["force"].reshape(8, 192, 3) - a["force"][None]).max() < 1e-10
    assert np.abs(b["virial"] - 8 * a["virial"]).max() < 1e-10 * np.abs(a["virial"]).max() * 8


def test_atom_rows_pieces_assemble_to_eval(water192_cond):
    """The sampled-row path used for the large configs: F_i = sum_k f_ik - sum_{(j,k): nlist[j][k]=i} f_jk."""
    cfg = water192_cond
    o = cfg["oracle"]
    full = o.eval(cfg["coord"], cfg["types"], cfg["box"])
    i = 57
    row = full["nlist"][i]
    nbrs = row[row >= 0]
    rows = np.concatenate([[i], nbrs])
    nl, _ = o.build_nlist(cfg["coord"], cfg["types"], cfg["box"], rows=rows)
    out = o.atom_rows(cfg["coord"], cfg["types"], cfg["box"], rows, nl)
    f = out["fslot"][0].sum(0)
    for q in range(1, len(rows)):
        hit = np.where(nl[q] == i)[0]
        assert len(hit) == 1
        f -= out["fslot"][q, hit[0]]
    assert np.abs(f - full["force"][i]).max() < 1e-12
    assert out["atom_energy"][0] == full["atom_energy"][i]


def test_atom_virial_is_minus_the_strain_derivative_of_each_atom_energy(water192_cond):
    """Per-atom virial, centre-atom split: Xi_i[a][b] = -sum_k d_ik[a] (dE_i/dd_ik)[b].  Under
    x -> (1 + eps) x every displacement of atom i's environment is strained, so dE_i/d eps_ab = -Xi_i[b][a]: pinned by
    central differences of E_i itself — diagonal strains of the periodic box, and all nine components on a cluster in a
    box far larger than it, where a shear of the coordinates needs no sheared box.  E_i is invariant under rotations of
    its environment, so every Xi_i is symmetric (checked): the index order cannot and need not be told apart."""
    cfg = water192_cond
    o, coord, types, box = cfg["oracle"], cfg["coord"], cfg["types"], cfg["box"]
    av = o.atom_virial(coord, types, box)
    ref = o.eval(coord, types, box)
    assert np.abs(av.sum(axis=0) - ref["virial"]).max() < 1e-11 * np.abs(ref["virial"]).max()
    assert np.abs(av - av.transpose(0, 2, 1)).max() < 1e-12 * np.abs(av).max()
    h = 1e-6
    for a in range(3):
        e = []
        for sgn in (+1, -1):
            F = np.eye(3)
            F[a, a] += sgn * h
            e.append(o.eval(coord @ F.T, types, (box.reshape(3, 3) @ F.T).reshape(9))["atom_energy"])
        fd = -(e[0] - e[1]) / (2 * h)
        assert np.abs(fd - av[:, a, a]).max() < 5e-7 * max(1.0, np.abs(fd).max())
    # cluster: 40 atoms of the same configuration in a 60 A box
    x = coord[:40] - coord[:40].mean(axis=0) + 30.0
    t = types[:40]
    big = np.diag([60.0, 60.0, 60.0]).reshape(9)
    avc = o.atom_virial(x, t, big)
    assert np.abs(avc).max() > 1e-3
    for a in range(3):
        for b in range(3):
            e = []
            for sgn in (+1, -1):
                F = np.eye(3)
                F[a, b] += sgn * h
                e.append(o.eval((x - 30.0) @ F.T + 30.0, t, big)["atom_energy"])
            fd = -(e[0] - e[1]) / (2 * h)                       # = -dE_i/d eps_ab = Xi_i[b][a]
            assert np.abs(fd - avc[:, b, a]).max() < 5e-7 * max(1.0, np.abs(fd).max()), (a, b)


def test_sampled_force_assembly_helper_matches_the_whole_evaluation():
    """conftest.oracle_forces_of (the reference of the 864,000-atom GPU parity tests) against dpo_eval on a small copper
    box: the forces and E_i of sampled atoms, assembled from per-row pieces, equal the whole evaluation's."""
    import gen
    from gen.weights import MODELS
    from oracle import Oracle
    from conftest import oracle_forces_of
    spec = MODELS["Cu32k"]
    coord, types, box = gen.copper_box(5, 0.05, seed=3)
    emb, fit = gen.make_weights(spec)
    fit = gen.condition_fit_w0(spec, fit)
    orc = Oracle.from_spec(spec, emb, fit)
    full = orc.eval(coord, types, box)
    atoms = np.array([0, 17, 250, 499])
    F, E, nl = oracle_forces_of(orc, coord, types, box, atoms)
    assert np.array_equal(nl, full["nlist"][atoms])
    assert np.abs(F - full["force"][atoms]).max() < 1e-13
    assert np.array_equal(E, full["atom_energy"][atoms])
