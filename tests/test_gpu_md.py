"""GPU tests of the molecular-dynamics driver dpb_md_run against the oracle's
velocity-Verlet driver, which is pinned by tests/test_oracle_md.py."""
import numpy as np
import pytest

import gen
from gen.weights import MODELS

pytestmark = pytest.mark.gpu


def _torch():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device (the library has no CPU fallback)")
    return torch


def _w192(conditioned=True):
    spec = MODELS["W192"]
    coord, types, box = gen.make_system("W192")
    emb, fit = gen.make_weights(spec)
    if conditioned:
        fit = gen.condition_fit_w0(spec, fit)
    vel = gen.maxwell_boltzmann(types, gen.MASSES["W192"], 330.0, seed=gen.SEED_BASE + 500)
    return spec, emb, fit, coord, types, box, vel


def _gpu_md(spec, emb, fit, coord, vel, types, box, mass, precision=0, **kw):
    torch = _torch()
    from paper_2004_11658_b200 import DPModel
    m = DPModel.from_spec(spec, emb, fit, precision=precision)
    dc, dv = torch.tensor(coord, device="cuda"), torch.tensor(vel, device="cuda")
    dt = torch.tensor(types, device="cuda")
    thermo, info = m.md_run(dc, dv, dt, mass, box, **kw)
    out = dc.cpu().numpy(), dv.cpu().numpy(), thermo, info
    m.close()
    return out


def test_md_trajectory_matches_oracle():
    """20 steps of 0.5 fs on the 192-atom water box: positions, velocities and every thermo row against the oracle."""
    from oracle import Oracle
    spec, emb, fit, coord, types, box, vel = _w192()
    mass = gen.MASSES["W192"]
    xr, vr, tr = Oracle.from_spec(spec, emb, fit).md_run(coord, vel, types, mass, box, 0.5, 20, thermo_every=5)
    x, v, th, info = _gpu_md(spec, emb, fit, coord, vel, types, box, mass, dt_fs=0.5, nsteps=20, thermo_every=5)
    assert info["n_thermo"] == 5 and info["n_rebuilds"] == 21
    assert np.abs(x - xr).max() <= 1e-10 and np.abs(v - vr).max() <= 1e-11
    assert np.abs(th[:, 0] - tr[:, 0]).max() <= 1e-10 * np.abs(tr[:, 0]).max()
    assert np.abs(th[:, 1] - tr[:, 1]).max() <= 1e-10 * np.abs(tr[:, 1]).max()
    assert abs(th[0, 2] - 330.0) < 1e-6
    assert np.abs(th[:, 3] - tr[:, 3]).max() <= 1e-9 * np.abs(tr[:, 3]).max()        # pressure (bar)


def test_md_energy_conservation_and_order():
    """NVE: |E_tot(t) - E_tot(0)| stays small against the kinetic-energy swing and drops ~4x when dt is halved."""
    spec, emb, fit, coord, types, box, vel = _w192()
    mass = gen.MASSES["W192"]
    devs, swing = [], 0.0
    for dt, n in ((0.5, 100), (0.25, 200)):
        _, _, th, _ = _gpu_md(spec, emb, fit, coord, vel, types, box, mass, dt_fs=dt, nsteps=n)
        etot = th[:, 0] + th[:, 1]
        devs.append(np.abs(etot - etot[0]).max())
        swing = np.ptp(th[:, 1])
    assert swing > 50 * devs[0]
    assert 2.5 < devs[0] / devs[1] < 6.0, devs


def test_md_skin_list_reuse_equals_fresh_search():
    """2 A skin, rebuilt every 50 steps (here every 20 of 60 steps, 1536 atoms so that r_c + skin < L/2).
    As long as no atom moves more than skin/2 the formatted list is the same list, so the trajectory agrees with the
    run that searches from the cell list at every step to rounding (the force scatter order differs)."""
    spec, emb, fit, coord, types, box, vel = _w192()
    coord, types8, box8 = gen.replicate(coord, types, box, 2)
    vel8 = np.tile(vel, (8, 1))
    mass = gen.MASSES["W192"]
    kw = dict(dt_fs=0.5, nsteps=60, thermo_every=20)
    x0, v0, th0, i0 = _gpu_md(spec, emb, fit, coord, vel8, types8, box8, mass, **kw)
    x1, v1, th1, i1 = _gpu_md(spec, emb, fit, coord, vel8, types8, box8, mass, rebuild_every=20, skin=2.0, **kw)
    assert i0["n_rebuilds"] == 61 and i1["n_rebuilds"] == 4
    assert not i1["skin_violated"] and 0.1 < i1["max_displacement"] < 1.0
    assert np.abs(x1 - x0).max() <= 1e-9 and np.abs(v1 - v0).max() <= 1e-10
    assert np.abs(th1 - th0).max() <= 1e-9 * np.abs(th0).max()
    # a skin that is far too small for the interval is reported
    _, _, _, i2 = _gpu_md(spec, emb, fit, coord, vel8, types8, box8, mass, rebuild_every=30, skin=0.05, **kw)
    assert i2["skin_violated"]


def test_md_mixed_precision_tracks_fp64():
    """DPB_TF32 forces (1e-3 eV/A bar) in the same integrator: after 20 steps the trajectory is within 1e-4 A of the
    fp64 one and the total energy is conserved to the same order."""
    spec, emb, fit, coord, types, box, vel = _w192()
    mass = gen.MASSES["W192"]
    kw = dict(dt_fs=0.5, nsteps=20)
    x0, v0, th0, _ = _gpu_md(spec, emb, fit, coord, vel, types, box, mass, **kw)
    x1, v1, th1, _ = _gpu_md(spec, emb, fit, coord, vel, types, box, mass, precision=1, **kw)
    assert np.abs(x1 - x0).max() <= 1e-4
    e0, e1 = th0[:, 0] + th0[:, 1], th1[:, 0] + th1[:, 1]
    assert np.abs(e1 - e1[0]).max() <= 3 * np.abs(e0 - e0[0]).max() + 1e-3
    # skin list in mixed precision (r_c + skin = 6.2 A < L/2 = 6.21 A): same trajectory as searching every step
    x2, v2, th2, i2 = _gpu_md(spec, emb, fit, coord, vel, types, box, mass, precision=1, rebuild_every=2, skin=0.2, **kw)
    assert i2["n_rebuilds"] == 11 and not i2["skin_violated"], i2
    # the skin grid sorts the atoms differently, so the 128-pair tiles (and their fp32 partial sums) differ: fp32-level
    assert np.abs(x2 - x1).max() <= 1e-6


def test_md_argument_errors():
    from paper_2004_11658_b200 import DPBError
    spec, emb, fit, coord, types, box, vel = _w192()
    mass = gen.MASSES["W192"]
    with pytest.raises(DPBError) as e:      # r_c + skin = 8 A >= L/2 = 6.21 A
        _gpu_md(spec, emb, fit, coord, vel, types, box, mass, dt_fs=0.5, nsteps=2, rebuild_every=2, skin=2.0)
    assert e.value.status == -2
    with pytest.raises(DPBError) as e:
        _gpu_md(spec, emb, fit, coord, vel, types, box, mass, dt_fs=-1.0, nsteps=2)
    assert e.value.status == -1


def test_decomposition_md_on_one_gpu_against_dpb_md_run():
    """dd.md_run with world size 1 on the device — libdpb's kick / drift / kinetic-energy kernels
    (binding.CudaIntegrator), migration across the periodic boundary, ghost images, dpb_eval_local, force fold-back —
    against dpb_md_run on the same box: positions (mod L), velocities, E_pot and E_kin after 20 steps.  Also the three
    integrator kernels against the formulas written in numpy."""
    import torch
    import paper_2004_11658_b200 as pk
    from paper_2004_11658_b200.binding import CudaIntegrator
    from paper_2004_11658_b200.dd import BrickDecomposition
    spec = MODELS["W192"]
    coord, types, box = gen.make_system("W192")
    emb, fit = gen.make_weights(spec)
    fit = gen.condition_fit_w0(spec, fit)
    masses = gen.MASSES["W192"]
    vel = gen.maxwell_boltzmann(types, masses, 330.0, seed=5) * 8.0
    m = pk.DPModel.from_spec(spec, emb, fit)
    dc, dv = torch.tensor(coord, device="cuda"), torch.tensor(vel, device="cuda")
    dt = torch.tensor(types, device="cuda")
    # integrator kernels against numpy
    integ = CudaIntegrator(masses, 0.5, dc.device)
    amu = 1.66053906660e-27 * 1e10 / 1.602176634e-19
    f = torch.tensor(np.random.default_rng(1).normal(size=coord.shape), device="cuda")
    x1, v1 = dc.clone(), dv.clone()
    integ.kick_drift(x1, v1, f, dt)
    mm = np.asarray(masses)[types] * amu
    v_ref = vel + (0.25 / mm)[:, None] * f.cpu().numpy()
    assert np.abs(v1.cpu().numpy() - v_ref).max() < 1e-14 and np.abs(x1.cpu().numpy() - (coord + 0.5 * v_ref)).max() < 1e-12
    integ.kick(v1, f, dt)
    assert np.abs(v1.cpu().numpy() - (v_ref + (0.25 / mm)[:, None] * f.cpu().numpy())).max() < 1e-14
    ek = integ.kinetic_energy(dv, dt).item()
    assert abs(ek - (0.5 * mm * (vel ** 2).sum(axis=1)).sum()) < 1e-12 * ek
    # the run
    xa, va = dc.clone(), dv.clone()
    thermo, info = m.md_run(xa, va, dt, masses, box, 0.5, 20, thermo_every=5)
    dd = BrickDecomposition(box, spec.rcut, grid=(1, 1, 1), rank=0, world=1)
    mask, w = dd.owned_mask(dc)
    tags = torch.arange(len(coord), device="cuda", dtype=torch.float64)
    xb, vb, tb, gb, th = dd.md_run(lambda x, t, nloc, bounds: m.eval_local(x, t, nloc, bounds, want_info=False), integ,
                                   w.contiguous().clone(), dv.clone(), dt, 20, thermo_every=5, tags=tags)
    torch.cuda.synchronize()
    order = gb.long()
    L = torch.tensor([box[0], box[4], box[8]], device="cuda")
    d = xb - xa[order]
    d -= torch.round(d / L) * L
    assert d.abs().max().item() < 1e-9 and (vb - va[order]).abs().max().item() < 1e-10
    assert torch.equal(tb, dt[order])
    th = th.cpu().numpy()
    assert np.abs(th[:, 0] - thermo[:, 0]).max() < 1e-10 * np.abs(thermo[:, 0]).max()
    assert np.abs(th[:, 1] - thermo[:, 1]).max() < 1e-10 * np.abs(thermo[:, 1]).max()
    m.close()
