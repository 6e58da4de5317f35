"""Domain decomposition (paper_2004_11658_b200/dd.py) on CPU:
world sizes 1, 2, 4 and 8 over gloo.  The per-brick evaluator here is the ORACLE's dpo_eval_local (tests may call the
oracle; the product passes DPModel.eval_local), so these tests cover exactly the host logic: brick ownership, the
three-stage forward exchange with periodic shifts, ghost forwarding to edges and corners, the reverse exchange that adds
the ghost forces to their owners, and the ten-double all-reduce.  Reference: the oracle's periodic evaluation."""
import os
import socket
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
sys.path.insert(0, os.path.join(ROOT, "tests"))


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


def _system():
    from conftest import small_model, random_box
    spec, emb, fit = small_model(ntypes=2, s1=4, m_axis=3, fit_width=8, sel=(20, 28), rcut=3.0, rcut_smth=0.8, seed=5,
                                 fit_scale=0.05)
    coord, types, box = random_box(90, 7.0, 2, seed=13, min_dist=1.1)
    box = np.array(box, dtype=np.float64).copy()
    box[0], box[4], box[8] = 7.0, 8.0, 9.5                         # anisotropic: a swapped dimension shows
    coord = np.random.default_rng(3).uniform(0.0, 1.0, size=coord.shape) * np.array([7.0, 8.0, 9.5])
    return spec, emb, fit, coord, types, box


def _oracle_evaluator(orc):
    def ev(x, t, nloc, bounds):
        xn, tn = x.numpy(), t.numpy()
        b = np.asarray(bounds)
        assert (xn >= b[:3] - 1e-12).all() and (xn <= b[3:] + 1e-12).all()        # what dpb_eval_local would check
        r = orc.eval_local(xn, tn, nloc, want_nlist=False)
        return {"energy": torch.tensor([r["energy"]], dtype=torch.float64), "atom_energy": torch.from_numpy(r["atom_energy"].copy()),
                "force": torch.from_numpy(r["force"].copy()), "virial": torch.from_numpy(r["virial"].copy())}
    return ev


def _run_rank(rank, world, grid):
    from oracle import Oracle
    from paper_2004_11658_b200.dd import BrickDecomposition
    spec, emb, fit, coord, types, box = _system()
    orc = Oracle.from_spec(spec, emb, fit)
    dd = BrickDecomposition(box, spec.rcut, grid=grid, rank=rank, world=world)
    mask, w = dd.owned_mask(torch.from_numpy(coord))
    ids = torch.nonzero(mask).flatten()
    out = dd.evaluate(_oracle_evaluator(orc), w[ids].contiguous(), torch.from_numpy(types.astype(np.int32))[ids])
    return ids.numpy(), out


def _reference():
    from oracle import Oracle
    spec, emb, fit, coord, types, box = _system()
    return Oracle.from_spec(spec, emb, fit).eval(coord, types, box, want_nlist=False), len(coord)


def _worker(rank, world, port, grid, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        ids, out = _run_rank(rank, world, grid)
        q.put((rank, ids, out["energy"].numpy(), out["virial"].numpy(), out["force"].numpy(),
               out["atom_energy"].numpy(), out["nall"]))
    finally:
        dist.destroy_process_group()


def _check(results, world):
    ref, n = _reference()
    F, Ei, seen = np.zeros((n, 3)), np.zeros(n), np.zeros(n, int)
    for rank, ids, e, vir, f, ei, nall in results:
        assert abs(e[0] - ref["energy"]) < 1e-12 * abs(ref["energy"])           # every rank holds the global E
        assert np.abs(vir - ref["virial"]).max() < 1e-11 * max(1.0, np.abs(ref["virial"]).max())
        F[ids] += f
        Ei[ids] = ei
        seen[ids] += 1
        assert nall > len(ids)                                                   # there are ghosts
    assert (seen == 1).all()                                                     # every atom has exactly one owner
    assert np.abs(F - ref["force"]).max() < 1e-12 * max(1.0, np.abs(ref["force"]).max())
    assert np.abs(Ei - ref["atom_energy"]).max() < 1e-12 * np.abs(ref["atom_energy"]).max()


def test_single_rank_periodic_images_only():
    """world 1: every ghost is a periodic image of a local atom; the exchange is a local copy."""
    ids, out = _run_rank(0, 1, (1, 1, 1))
    _check([(0, ids, out["energy"].numpy(), out["virial"].numpy(), out["force"].numpy(), out["atom_energy"].numpy(),
             out["nall"])], 1)


@pytest.mark.parametrize("world,grid", [(2, (2, 1, 1)), (2, (1, 1, 2)), (4, (2, 2, 1)), (8, (2, 2, 2)), (3, (1, 1, 3))])
def test_bricks_over_gloo(world, grid):
    """2 bricks in a dimension (both neighbours are the same rank: two messages per pair, matched in order), 3 bricks
    (distinct neighbours), and 2 x 2 x 2 (corner ghosts travel through three stages and their forces three stages back)."""
    port = _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, grid, q)) for r in range(world)]
    for p in procs:
        p.start()
    results = [q.get(timeout=240) for _ in range(world)]
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    _check(sorted(results, key=lambda r: r[0]), world)


def test_grid_choice_and_refusals():
    from paper_2004_11658_b200.dd import BrickDecomposition, choose_grid
    assert choose_grid(8, (10.0, 10.0, 10.0)) == (2, 2, 2)
    assert choose_grid(2, (10.0, 20.0, 10.0)) == (1, 2, 1)
    assert choose_grid(6, (30.0, 20.0, 10.0)) == (3, 2, 1)
    box = np.diag([7.0, 8.0, 9.5]).reshape(-1)
    with pytest.raises(ValueError):
        BrickDecomposition(box, 3.0, grid=(3, 1, 1), rank=0, world=3)            # 7 / 3 < r_c
    with pytest.raises(ValueError):
        BrickDecomposition(box, 3.0, grid=(2, 1, 1), rank=0, world=4)
    d = BrickDecomposition(box, 3.0, grid=(1, 2, 3), rank=5, world=6)
    assert d.index == (0, 1, 2) and d.neighbour(2, +1) == d.rank_of((0, 1, 0)) == 3 and d.neighbour(1, -1) == 2
    assert np.allclose(d.bounds(), [-3.0, 1.0, 9.5 * 2 / 3 - 3.0, 10.0, 11.0, 12.5])


# ---- molecular dynamics on the decomposition: migration + time loop against the oracle's single-box MD --------------
MASS2 = (15.999, 1.008)
AMU = 1.66053906660e-27 * 1e10 / 1.602176634e-19           # 1 amu A^2/fs^2 in eV, straight from CODATA 2018


class _TorchIntegrator:
    """Test-side velocity-Verlet pieces on CPU tensors (the product's are libdpb kernels, binding.CudaIntegrator)."""

    def __init__(self, masses, dt):
        self.m = torch.tensor(masses, dtype=torch.float64) * AMU
        self.dt = dt

    def kick_drift(self, coord, vel, force, types):
        vel += (0.5 * self.dt / self.m[types.long()])[:, None] * force
        coord += self.dt * vel

    def kick(self, vel, force, types):
        vel += (0.5 * self.dt / self.m[types.long()])[:, None] * force

    def kinetic_energy(self, vel, types):
        return (0.5 * self.m[types.long()] * (vel ** 2).sum(dim=1)).sum().reshape(1)


def _md_inputs():
    import gen
    spec, emb, fit, coord, types, box = _system()
    vel = gen.maxwell_boltzmann(types, MASS2, 330.0, seed=21) * 12.0          # fast: atoms cross brick faces in 12 steps
    return spec, emb, fit, coord, types, box, vel


def _md_rank(rank, world, grid, nsteps, dt):
    from oracle import Oracle
    from paper_2004_11658_b200.dd import BrickDecomposition
    spec, emb, fit, coord, types, box, vel = _md_inputs()
    orc = Oracle.from_spec(spec, emb, fit)
    dd = BrickDecomposition(box, spec.rcut, grid=grid, rank=rank, world=world)
    mask, w = dd.owned_mask(torch.from_numpy(coord))
    ids = torch.nonzero(mask).flatten()
    x, v, t, tags, thermo = dd.md_run(_oracle_evaluator(orc), _TorchIntegrator(MASS2, dt), w[ids].contiguous().clone(),
                                      torch.from_numpy(vel)[ids].contiguous().clone(),
                                      torch.from_numpy(types.astype(np.int32))[ids], nsteps, thermo_every=4,
                                      tags=ids.to(torch.float64))
    return tags.numpy().astype(np.int64), x.numpy(), v.numpy(), t.numpy(), thermo.numpy(), ids.numpy()


def _md_worker(rank, world, port, grid, nsteps, dt, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        q.put((rank,) + _md_rank(rank, world, grid, nsteps, dt))
    finally:
        dist.destroy_process_group()


def _md_check(results, nsteps, dt):
    from oracle import Oracle
    spec, emb, fit, coord, types, box, vel = _md_inputs()
    xr, vr, th = Oracle.from_spec(spec, emb, fit).md_run(coord, vel, types, MASS2, box, dt, nsteps, thermo_every=4)
    L = np.array([box[0], box[4], box[8]])
    n = len(coord)
    seen, moved = np.zeros(n, int), 0
    for rank, tags, x, v, t, thermo, n0 in results:
        seen[tags] += 1
        d = x - xr[tags]
        d -= np.round(d / L) * L                                  # the decomposition keeps atoms wrapped, the oracle does not
        assert np.abs(d).max() < 1e-9
        assert np.abs(v - vr[tags]).max() < 1e-10
        assert np.array_equal(t, types[tags])
        assert np.abs(thermo[:, 0] - th[:, 0]).max() < 1e-10 * np.abs(th[:, 0]).max()      # E_pot, on every rank
        assert np.abs(thermo[:, 1] - th[:, 1]).max() < 1e-10 * np.abs(th[:, 1]).max()      # E_kin
        moved += len(set(tags.tolist()) - set(n0.tolist()))       # atoms this rank received during the run
    assert (seen == 1).all()
    return moved


def test_md_single_rank_against_the_oracle():
    res = (0,) + _md_rank(0, 1, (1, 1, 1), 12, 1.0)
    _md_check([res], 12, 1.0)


@pytest.mark.parametrize("world,grid", [(2, (1, 1, 2)), (4, (2, 2, 1))])
def test_md_with_migration_over_gloo(world, grid):
    """Atoms cross brick faces and the periodic boundary during the run: positions (mod L), velocities, types and the
    global E_pot / E_kin of every rank against the oracle's single-box velocity-Verlet, atom by atom through the tags."""
    port = _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_md_worker, args=(r, world, port, grid, 12, 1.0, q)) for r in range(world)]
    for p in procs:
        p.start()
    results = [q.get(timeout=400) for _ in range(world)]
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    moved = _md_check(sorted(results, key=lambda r: r[0]), 12, 1.0)
    assert moved > 0                                             # the run did exercise the migration
