"""Pins for the oracle's sub-region evaluation with explicit ghost atoms (dpo_eval_local; SURVEY.md §8(e) / §8(f) NEXT #2,
#3).  None of them retypes its arithmetic: the partition identity against the (separately pinned)
periodic evaluation, a finite-difference check of the force on a GHOST atom (the term the reverse exchange carries,
PAPER.md:149), an isolated cluster against the periodic code in a box far larger than the cluster, and the degenerate
cases.  The ghost shells here are built by brute force over the 27 periodic images.  No CUDA."""
import itertools

import numpy as np

from oracle import Oracle

from conftest import small_model, random_box


def brute_force_domain(coord, box, lo, hi, rc):
    """Local atoms: wrapped position inside [lo, hi).  Ghosts: every periodic image (27 shifts) of every atom that is not
    the local copy itself and lies within rc of the brick (distance to the brick, a superset of what is needed).
    Returns (local indices, ghost owner indices, ghost coordinates)."""
    L = np.array([box[0], box[4], box[8]])
    w = coord - np.floor(coord / L) * L
    loc = np.nonzero(np.all((w >= lo) & (w < hi), axis=1))[0]
    is_loc = np.zeros(len(coord), bool)
    is_loc[loc] = True
    owners, xyz = [], []
    for s in itertools.product((-1, 0, 1), repeat=3):
        x = w + np.array(s) * L
        gap = np.maximum(np.maximum(lo - x, x - hi), 0.0)
        near = (gap ** 2).sum(axis=1) <= rc * rc
        if s == (0, 0, 0):
            near &= ~is_loc
        idx = np.nonzero(near)[0]
        owners.append(idx)
        xyz.append(x[idx])
    return loc, np.concatenate(owners), np.concatenate(xyz), w


def bricks(box, grid):
    L = np.array([box[0], box[4], box[8]])
    for ix in itertools.product(*(range(g) for g in grid)):
        lo = L * np.array(ix) / np.array(grid)
        hi = L * (np.array(ix) + 1) / np.array(grid)
        yield lo, hi


def _setup(n=60, L=9.5, seed=3):
    spec, emb, fit = small_model(ntypes=2, s1=4, m_axis=3, fit_width=8, sel=(20, 28), rcut=4.0, rcut_smth=1.0,
                                 seed=5, fit_scale=0.05)
    coord, types, box = random_box(n, L, 2, seed=seed, min_dist=1.3)
    return spec, emb, fit, coord, types, box


def _sum_over_domains(o, coord, types, box, grid, rc):
    n = len(coord)
    E, F, V, Ei = 0.0, np.zeros((n, 3)), np.zeros((3, 3)), np.full(n, np.nan)
    nl_owner = {}
    seen = 0
    for lo, hi in bricks(box, grid):
        loc, own, gxyz, w = brute_force_domain(coord, box, lo, hi, rc)
        seen += len(loc)
        x = np.concatenate([w[loc], gxyz])
        t = np.concatenate([types[loc], types[own]])
        r = o.eval_local(x, t, len(loc))
        E += r["energy"]
        V += r["virial"]
        ids = np.concatenate([loc, own])
        np.add.at(F, ids, r["force"])                     # the reverse exchange: ghost increments go to the owner
        Ei[loc] = r["atom_energy"]
        for q, i in enumerate(loc):
            row = r["nlist"][q]
            nl_owner[i] = np.where(row >= 0, ids[np.maximum(row, 0)], -1)
    assert seen == n
    return E, Ei, F, V, nl_owner


def test_partition_identity_against_the_periodic_evaluation():
    """E, E_i, F and the virial of the periodic box = the sums over its sub-regions (2, 4 and 8 bricks, and the
    one-brick case in which every ghost is a periodic image of a local atom).  Dropping the ghost forces, summing E_i
    over ghosts too, or a virial that leaves out local-ghost pairs all break it."""
    spec, emb, fit, coord, types, box = _setup()
    o = Oracle.from_spec(spec, emb, fit)
    ref = o.eval(coord, types, box)
    for grid in ((1, 1, 1), (2, 1, 1), (1, 2, 2), (2, 2, 2)):
        E, Ei, F, V, nl_owner = _sum_over_domains(o, coord, types, box, grid, spec.rcut)
        assert abs(E - ref["energy"]) < 1e-12 * abs(ref["energy"]), grid
        assert np.abs(Ei - ref["atom_energy"]).max() < 1e-12 * np.abs(ref["atom_energy"]).max()
        assert np.abs(F - ref["force"]).max() < 1e-12 * max(1.0, np.abs(ref["force"]).max())
        assert np.abs(V - ref["virial"]).max() < 1e-11 * max(1.0, np.abs(ref["virial"]).max())
        # the formatted list names the same neighbours (as owners), slot by slot, except where two images tie exactly
        same = sum(np.array_equal(nl_owner[i], ref["nlist"][i]) for i in range(len(coord)))
        assert same == len(coord)


def test_force_on_a_ghost_atom_is_minus_the_gradient_of_the_local_energy():
    """Central differences of E_local with respect to a ghost coordinate: pins the sign and the presence of the ghost
    part of the force (it has to be sent back, it is not minus the local part)."""
    spec, emb, fit, coord, types, box = _setup()
    o = Oracle.from_spec(spec, emb, fit)
    lo, hi = next(iter(bricks(box, (2, 1, 1))))
    loc, own, gxyz, w = brute_force_domain(coord, box, lo, hi, spec.rcut)
    x = np.concatenate([w[loc], gxyz])
    t = np.concatenate([types[loc], types[own]])
    r = o.eval_local(x, t, len(loc))
    g = len(loc) + int(np.argmax(np.abs(r["force"][len(loc):]).sum(axis=1)))   # the ghost that feels the most
    assert np.abs(r["force"][g]).max() > 1e-6
    h = 1e-5
    for c in range(3):
        xp, xm = x.copy(), x.copy()
        xp[g, c] += h
        xm[g, c] -= h
        d = (o.eval_local(xp, t, len(loc))["energy"] - o.eval_local(xm, t, len(loc))["energy"]) / (2 * h)
        assert abs(-d - r["force"][g, c]) < 1e-7 * max(1.0, abs(d))
    # local atom too
    i = 0
    for c in range(3):
        xp, xm = x.copy(), x.copy()
        xp[i, c] += h
        xm[i, c] -= h
        d = (o.eval_local(xp, t, len(loc))["energy"] - o.eval_local(xm, t, len(loc))["energy"]) / (2 * h)
        assert abs(-d - r["force"][i, c]) < 1e-7 * max(1.0, abs(d))


def test_isolated_cluster_equals_the_periodic_code_in_a_large_box():
    """nloc = nall, a cluster of diameter < 10 A: the periodic evaluation in a 60 A box sees no image either."""
    spec, emb, fit, coord, types, box = _setup(n=40, L=9.0, seed=8)
    o = Oracle.from_spec(spec, emb, fit)
    big = np.diag([60.0, 60.0, 60.0]).reshape(-1)
    x = coord + 25.0
    a = o.eval_local(x, types, len(x))
    b = o.eval(x, types, big)
    assert np.array_equal(a["nlist"], b["nlist"])
    assert abs(a["energy"] - b["energy"]) < 1e-13 * abs(b["energy"])
    assert np.abs(a["force"] - b["force"]).max() < 1e-13 * max(1.0, np.abs(b["force"]).max())
    assert np.abs(a["virial"] - b["virial"]).max() < 1e-12 * max(1.0, np.abs(b["virial"]).max())
    assert np.abs(a["force"].sum(axis=0)).max() < 1e-12            # no ghosts: momentum is conserved


def test_degenerate_cases():
    spec, emb, fit, coord, types, box = _setup(n=20, L=9.0, seed=2)
    o = Oracle.from_spec(spec, emb, fit)
    r = o.eval_local(coord, types, 0)                               # ghosts only: nothing to evaluate
    assert r["energy"] == 0.0 and not r["force"].any() and not r["virial"].any()
    one = o.eval_local(coord[:1], types[:1], 1)                     # a lone atom: E_i of an empty environment, F = 0
    far = o.eval_local(np.array([[0.0, 0, 0], [50.0, 0, 0]]), np.array([0, 0], dtype=np.int32), 2)
    t0 = o.eval_local(np.array([[1.0, 2, 3]]), np.array([0], dtype=np.int32), 1)
    assert not one["force"].any() and (one["nlist"] == -1).all()
    assert abs(far["energy"] - 2 * t0["energy"]) < 1e-15 * max(1.0, abs(t0["energy"]))
    # ghosts beyond r_c of every local atom change nothing
    x = np.concatenate([coord, coord[:5] + 40.0])
    t = np.concatenate([types, types[:5]])
    a, b = o.eval_local(coord, types, len(coord)), o.eval_local(x, t, len(coord))
    assert a["energy"] == b["energy"] and np.array_equal(a["force"], b["force"][:len(coord)])
    assert not b["force"][len(coord):].any()


# ---- general periodic cells through explicit images (paper_2004_11658_b200/cell.py) ----------
def _brute_images(coord, cell, rc, shells=2):
    """Every lattice image (|n_c| <= shells) that has some atom of the cell within rc: O(N^2), independent of cell.py."""
    a = np.asarray(cell).reshape(3, 3)
    s = coord @ np.linalg.inv(a)
    w = (s - np.floor(s)) @ a
    xs, own = [w], [np.arange(len(w))]
    for n in itertools.product(range(-shells, shells + 1), repeat=3):
        if n == (0, 0, 0):
            continue
        x = w + np.array(n) @ a
        d2 = ((x[:, None, :] - w[None, :, :]) ** 2).sum(-1).min(axis=1)
        idx = np.nonzero(d2 <= rc * rc)[0]
        xs.append(x[idx])
        own.append(idx)
    return np.concatenate(xs), np.concatenate(own)


def _eval_cell_with_oracle(o, coord, types, cell, rc, images):
    x, own = images(coord, cell, rc)
    r = o.eval_local(x, types[own], len(coord), want_nlist=False)
    f = np.zeros((len(coord), 3))
    np.add.at(f, own, r["force"])
    return r["energy"], r["atom_energy"], f, r["virial"], len(x)


def _cell_heights(cell):
    """Perpendicular heights h_c = V / |a_j x a_k| of the parallelepiped spanned by the rows of `cell`."""
    a = np.asarray(cell, dtype=np.float64).reshape(3, 3)
    vol = abs(np.linalg.det(a))
    return np.array([vol / np.linalg.norm(np.cross(a[(c + 1) % 3], a[(c + 2) % 3])) for c in range(3)])


def _margin_images(coord, cell, rc):
    """The image selection rule of dpb_eval_cell (include/dpb.h, csrc/cell.cu), restated in numpy so that the RULE is
    pinned here without a GPU: wrap the fractional coordinates into [0, 1); keep every lattice image whose fractional
    coordinate t_c lies in [-r_c / h_c, 1 + r_c / h_c] for all c (ceil(r_c / h_c) shells per lattice direction); the
    bounds are the corners of the widened parallelepiped."""
    import itertools
    a = np.asarray(cell, dtype=np.float64).reshape(3, 3)
    h = _cell_heights(a)
    s = coord @ np.linalg.inv(a)
    s = s - np.floor(s)
    m = rc / h
    n = [int(np.ceil(v)) for v in m]
    parts, owners = [s], [np.arange(len(coord))]
    for shift in itertools.product(*(range(-k, k + 1) for k in n)):
        if shift == (0, 0, 0):
            continue
        t = s + np.array(shift, dtype=np.float64)
        idx = np.nonzero(((t >= -m) & (t <= 1.0 + m)).all(axis=1))[0]
        parts.append(t[idx])
        owners.append(idx)
    x = np.concatenate(parts) @ a
    corners = np.array([[(-m[c] if (k >> c) & 1 == 0 else 1.0 + m[c]) for c in range(3)] for k in range(8)]) @ a
    pad = 1e-9 * (1.0 + np.abs(corners).max())
    assert (x >= corners.min(axis=0) - pad).all() and (x <= corners.max(axis=0) + pad).all()   # the bounds hold them all
    return x, np.concatenate(owners)


def test_sheared_description_of_an_orthorhombic_lattice():
    """The cells (a1, a2, a3), (a1, a2 + a1, a3) and (a1, a2 + a1, a3 + a2 - a1) generate the same lattice, so E, E_i,
    F and the virial from explicit images of the sheared (triclinic) cells must equal the orthorhombic periodic
    evaluation; both image builders (brute force here, dpb_eval_cell's fractional-coordinate margins) are checked."""
    spec, emb, fit, coord, types, box = _setup()
    o = Oracle.from_spec(spec, emb, fit)
    ref = o.eval(coord, types, box)
    a = np.asarray(box).reshape(3, 3)
    cells = [a, np.array([a[0], a[1] + a[0], a[2]]), np.array([a[0], a[1] + a[0], a[2] + a[1] - a[0]])]
    for cell in cells:
        for images in (_brute_images, _margin_images):
            E, Ei, F, V, nall = _eval_cell_with_oracle(o, coord, types, cell, spec.rcut, images)
            assert abs(E - ref["energy"]) < 1e-12 * abs(ref["energy"])
            assert np.abs(Ei - ref["atom_energy"]).max() < 1e-12 * np.abs(ref["atom_energy"]).max()
            assert np.abs(F - ref["force"]).max() < 1e-11 * max(1.0, np.abs(ref["force"]).max())
            assert np.abs(V - ref["virial"]).max() < 1e-10 * max(1.0, np.abs(ref["virial"]).max())


def test_cell_images_thin_cell_and_heights():
    """dpb_eval_cell's image rule against the brute-force images on a genuinely triclinic cell thinner than 2 r_c in one
    direction (two image shells there), and the perpendicular heights of a sheared cell."""
    cell_heights = _cell_heights
    spec, emb, fit, coord, types, box = _setup(n=30, L=9.0, seed=6)
    o = Oracle.from_spec(spec, emb, fit)
    cell = np.array([[9.0, 0.0, 0.0], [2.5, 8.0, 0.0], [1.0, -1.5, 3.6]])     # height along c: 3.6 < r_c = 4
    assert np.allclose(cell_heights(cell), [9.0 * 8.0 * 3.6 / np.linalg.norm(np.cross(cell[1], cell[2])),
                                            9.0 * 8.0 * 3.6 / np.linalg.norm(np.cross(cell[2], cell[0])), 3.6])
    rng = np.random.default_rng(8)
    x = rng.uniform(0, 1, size=(30, 3)) @ cell
    a = _eval_cell_with_oracle(o, x, types, cell, spec.rcut, _brute_images)
    b = _eval_cell_with_oracle(o, x, types, cell, spec.rcut, _margin_images)
    assert b[4] >= a[4]                                             # the margin rule keeps a superset of the needed images
    assert abs(a[0] - b[0]) < 1e-12 * abs(a[0]) and np.abs(a[2] - b[2]).max() < 1e-11 and np.abs(a[3] - b[3]).max() < 1e-10
    assert np.abs(b[2].sum(axis=0)).max() < 1e-10                   # periodic system: total force vanishes
