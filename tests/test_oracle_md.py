"""Pins for the oracle's molecular-dynamics driver (velocity-Verlet NVE).
Nothing here compares the oracle with itself through the same formula: free flight (closed form), the order of the
integrator (error ~ dt^2), time reversibility, momentum conservation, and the unit constants from CODATA.  No CUDA."""
import numpy as np

import gen
from oracle import Oracle

from conftest import small_model, random_box

MASS2 = (15.999, 1.008)


def _setup(n=36, L=9.0, seed=4, T0=330.0):
    spec, emb, fit = small_model(ntypes=2, s1=4, m_axis=3, fit_width=8, sel=(16, 24), rcut=4.0, rcut_smth=1.0,
                                 seed=9, fit_scale=0.05)
    coord, types, box = random_box(n, L, 2, seed=seed, min_dist=1.4)
    vel = gen.maxwell_boltzmann(types, MASS2, T0, seed=77)
    return spec, emb, fit, coord, types, box, vel


def test_units_and_initial_temperature():
    """E_kin = 1/2 sum m v^2 in eV needs 1 amu A^2/fs^2 = m_u 1e10 / e (CODATA 2018: 103.6427 eV) and
    T = 2 E_kin / (3 N k_B): velocities rescaled to exactly 330 K by the generator (its own constants, straight from
    CODATA) must read 330 K in the oracle's thermo output."""
    spec, emb, fit, coord, types, box, vel = _setup()
    o = Oracle.from_spec(spec, emb, fit)
    _, _, th = o.md_run(coord, vel, types, MASS2, box, 0.5, 0)
    assert abs(th[0, 2] - 330.0) < 1e-6
    m = np.asarray(MASS2)[types]
    ek = 0.5 * (m[:, None] * vel ** 2).sum() * (1.66053906660e-27 * 1e10 / 1.602176634e-19)
    assert abs(th[0, 1] - ek) < 1e-9 * ek
    assert abs(th[0, 0] - o.eval(coord, types, box)["energy"]) < 1e-12 * abs(th[0, 0])


def test_free_flight_closed_form():
    """Weights that make E constant (everything zero except the output bias) => F = 0: x(t) = x0 + t v0 exactly in
    form, also for atoms that leave the box (coordinates are not wrapped), E_pot and E_kin constant."""
    spec, emb, fit, coord, types, box, vel = _setup()
    fit0 = np.zeros_like(fit)
    from gen.weights import fit_net_size
    per = fit_net_size(spec.dim_descrpt, spec.fit_width)
    fit0[per - 1] = 0.7
    fit0[2 * per - 1] = -0.2
    o = Oracle.from_spec(spec, np.zeros_like(emb), fit0)
    vel = vel * 40.0                                   # fast: many atoms cross the boundary in 50 steps
    x, v, th = o.md_run(coord, vel, types, MASS2, box, 0.5, 50, thermo_every=10)
    assert np.array_equal(v, vel)
    assert np.abs(x - (coord + 25.0 * vel)).max() < 1e-12
    assert (x < 0).any() or (x > box[0]).any()
    e0 = 0.7 * (types == 0).sum() - 0.2 * (types == 1).sum()
    assert np.abs(th[:, 0] - e0).max() < 1e-12 and np.ptp(th[:, 1]) < 1e-12 * th[0, 1]


def test_energy_conservation_is_second_order():
    """NVE with F = -grad E: the total-energy error of velocity-Verlet is bounded and ~ dt^2: halving dt divides the
    maximum deviation by ~4.  A wrong force sign, a missing half kick or a wrong mass factor all break this."""
    spec, emb, fit, coord, types, box, vel = _setup()
    o = Oracle.from_spec(spec, emb, fit)
    devs = []
    for dt, n in ((1.0, 40), (0.5, 80), (0.25, 160)):
        _, _, th = o.md_run(coord, vel, types, MASS2, box, dt, n)
        etot = th[:, 0] + th[:, 1]
        devs.append(np.abs(etot - etot[0]).max())
    assert np.ptp(th[:, 1]) > 100 * devs[-1]            # the kinetic energy really changes: forces act
    assert 2.5 < devs[0] / devs[1] < 6.0 and 2.5 < devs[1] / devs[2] < 6.0, devs


def test_time_reversibility_and_momentum():
    spec, emb, fit, coord, types, box, vel = _setup()
    o = Oracle.from_spec(spec, emb, fit)
    x1, v1, _ = o.md_run(coord, vel, types, MASS2, box, 0.5, 30)
    m = np.asarray(MASS2)[types][:, None]
    assert np.abs((m * v1).sum(0) - (m * vel).sum(0)).max() < 1e-12          # sum F = 0 at every step
    assert np.abs(x1 - coord).max() > 1e-2
    x2, v2, _ = o.md_run(x1, -v1, types, MASS2, box, 0.5, 30)
    assert np.abs(x2 - coord).max() < 1e-9 and np.abs(v2 + vel).max() < 1e-10


def test_one_step_against_hand_written_update():
    """One step written out with the oracle's own force evaluations (pins the order kick-drift-force-kick)."""
    spec, emb, fit, coord, types, box, vel = _setup()
    o = Oracle.from_spec(spec, emb, fit)
    dt = 0.5
    m = np.asarray(MASS2)[types][:, None] * gen.AMU_A2_FS2_IN_EV
    f0 = o.eval(coord, types, box)["force"]
    vh = vel + 0.5 * dt * f0 / m
    x1 = coord + dt * vh
    f1 = o.eval(x1, types, box)["force"]
    v1 = vh + 0.5 * dt * f1 / m
    x, v, th = o.md_run(coord, vel, types, MASS2, box, dt, 1)
    assert np.abs(x - x1).max() < 1e-13 and np.abs(v - v1).max() < 1e-13


def test_pressure_ideal_gas_and_virial_part():
    """thermo column 3 = P in bar (PAPER.md:298 lists the pressure among the thermo data).  Zero-force model: the ideal
    gas law P V = N k_B T with CODATA constants (1 eV/A^3 = e / 1e-30 m^3 = 1.602176634e11 Pa).  Atoms at rest: the
    virial part alone, P = -dE/dV, by central differences of the oracle's energy under an isotropic scaling."""
    spec, emb, fit, coord, types, box, vel = _setup()
    from gen.weights import fit_net_size
    per = fit_net_size(spec.dim_descrpt, spec.fit_width)
    fit0 = np.zeros_like(fit)
    fit0[per - 1] = 0.3
    o0 = Oracle.from_spec(spec, np.zeros_like(emb), fit0)
    _, _, th = o0.md_run(coord, vel, types, MASS2, box, 0.5, 0)
    V = box[0] * box[4] * box[8]
    p_ideal = len(types) * (1.380649e-23 / 1.602176634e-19) * 330.0 / V * (1.602176634e-19 / 1e-30 / 1e5)
    assert abs(th[0, 3] - p_ideal) < 1e-9 * p_ideal

    o = Oracle.from_spec(spec, emb, fit)
    _, _, th = o.md_run(coord, np.zeros_like(vel), types, MASS2, box, 0.5, 0)
    h = 1e-5
    e = []
    for s in (1 + h, 1 - h):
        e.append(o.eval(coord * s, types, box * s)["energy"])
    dEdV = (e[0] - e[1]) / (V * ((1 + h) ** 3 - (1 - h) ** 3))
    p_fd = -dEdV * 1.602176634e6
    assert abs(th[0, 3] - p_fd) < 1e-6 * max(1.0, abs(p_fd)), (th[0, 3], p_fd)
