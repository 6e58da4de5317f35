"""Closed-form and special-case pins for the oracle's per-stage functions (switch, env matrix, embedding,
descriptor, fitting).  No CUDA here."""
import numpy as np

import gen
from gen.weights import ModelSpec, emb_net_size, fit_net_size
from oracle import Oracle

from conftest import small_model


def test_switch_function_pins(water192):
    o = water192["oracle"]                       # rcs = 0.5, rc = 6.0
    assert o.switch(0.3) == (1.0, 0.0)           # w = 1 below rcs  => s = 1/r there
    assert o.switch(0.5)[0] == 1.0               # continuity at rcs
    assert o.switch(6.0) == (0.0, 0.0) and o.switch(7.0) == (0.0, 0.0)
    mid = 0.5 * (0.5 + 6.0)
    assert abs(o.switch(mid)[0] - 0.5) < 1e-15   # u = 1/2: 1 + (1/8)(-6/4 + 15/2 - 10) = 1/2
    # C^2 at both ends: w, w', w'' -> (1,0,0) at rcs and (0,0,0) at rc
    for r0, w0 in ((0.5, 1.0), (6.0, 0.0)):
        h = 1e-4
        side = +1 if r0 == 0.5 else -1
        w1, d1 = o.switch(r0 + side * h)
        assert abs(w1 - w0) < 1e-9 and abs(d1) < 1e-6          # w - w0 = O(h^3), w' = O(h^2)
    # dw is the derivative of w (central differences), monotone decay
    rs = np.linspace(0.6, 5.9, 40)
    for r in rs:
        h = 1e-6
        fd = (o.switch(r + h)[0] - o.switch(r - h)[0]) / (2 * h)
        assert abs(fd - o.switch(r)[1]) < 1e-8
        assert o.switch(r)[1] < 0


def test_displacement_minimum_image(water192):
    o = water192["oracle"]
    L = np.array([10.0, 12.0, 14.0])
    d, r = o.displacement([1.0, 1.0, 1.0], [9.5, 11.5, 1.5], L)
    assert np.allclose(d, [-1.5, -1.5, 0.5], atol=1e-15) and abs(r - np.sqrt(4.75)) < 1e-15
    d, r = o.displacement([1.0, 1.0, 1.0], [31.0, -23.0, 1.0], L)      # raw coordinates, several images away
    assert np.allclose(d, [0.0, 0.0, 0.0], atol=1e-14)
    d1, r1 = o.displacement([0.1, 0.2, 0.3], [3.3, 2.2, 1.1], L)
    d2, r2 = o.displacement([3.3, 2.2, 1.1], [0.1, 0.2, 0.3], L)
    assert np.array_equal(d1, -d2) and r1 == r2                        # exactly antisymmetric


def test_env_row_closed_form():
    """One pair: R~ = s (1, d/r) with s = w(r)/r (Eq. 5); padded slots are zero rows."""
    spec, emb, fit = small_model(ntypes=1, sel=(4,), rcut=4.0, rcut_smth=1.0)
    o = Oracle.from_spec(spec, emb, fit)
    box = np.diag([20.0] * 3).reshape(9)
    for dvec in ([0.6, 0.0, 0.0], [1.0, 2.0, -2.0], [0.0, 0.0, 3.9]):
        coord = np.array([[5.0, 5.0, 5.0], np.array([5.0, 5.0, 5.0]) + dvec])
        types = np.zeros(2, dtype=np.int32)
        nl, _ = o.build_nlist(coord, types, box)
        assert nl[0].tolist() == [1, -1, -1, -1]
        env, denv, disp = o.env_row(coord, types, box, 0, nl[0])
        r = np.linalg.norm(dvec)
        w = 1.0 if r < 1.0 else (lambda u: u ** 3 * (-6 * u * u + 15 * u - 10) + 1)((r - 1.0) / 3.0)
        s = w / r
        assert np.allclose(env[0], [s, s * dvec[0] / r, s * dvec[1] / r, s * dvec[2] / r], rtol=1e-14, atol=1e-16)
        assert np.all(env[1:] == 0) and np.all(denv[1:] == 0)
        assert np.allclose(disp[0], dvec, atol=1e-15)
        # below rcs: s = 1/r exactly in form
        if r < 1.0:
            assert abs(env[0, 0] - 1.0 / r) < 1e-15
        # denv = d env / d d  (central differences on the displacement)
        h = 1e-6
        for c in range(3):
            cp, cm = coord.copy(), coord.copy()
            cp[1, c] += h
            cm[1, c] -= h
            ep, _, _ = o.env_row(cp, types, box, 0, nl[0])
            em, _, _ = o.env_row(cm, types, box, 0, nl[0])
            assert np.allclose((ep[0] - em[0]) / (2 * h), denv[0, :, c], atol=2e-8)


def test_embedding_concat_pin():
    """Zero W1, W2, b1, b2  =>  g = [h0 || h0 || h0 || h0] with h0 = tanh(x W0 + b0): pins that (x, x) in Eq. 9
    is concatenation (Eq. 12 :268) and that layer 0 has no skip (Eq. 8)."""
    s1 = 5
    spec = ModelSpec("t", 1, 4.0, 1.0, (4,), s1, 2, 6, 0)
    emb, fit = gen.make_weights(spec, seed=3)
    emb = emb.copy()
    emb[2 * s1:] = 0.0                               # keep W0, b0 only
    o = Oracle.from_spec(spec, emb, fit)
    for x in (-1.3, 0.0, 0.37, 2.5):
        h0 = np.tanh(x * emb[:s1] + emb[s1:2 * s1])
        assert np.allclose(o.embed(0, 0, x), np.tile(h0, 4), rtol=0, atol=1e-15)
    o0 = Oracle.from_spec(spec, np.zeros_like(emb), fit)
    assert np.all(o0.embed(0, 0, 0.7) == 0.0)         # all-zero weights => g = 0


def test_embedding_against_numpy_matmul():
    """The general case against a numpy restatement with library matmuls (A @ W), per net (a, t)."""
    spec, emb, fit = small_model(ntypes=2, s1=6)
    o = Oracle.from_spec(spec, emb, fit)
    s1 = spec.emb_s1
    for a in range(2):
        for t in range(2):
            p = emb[(a * 2 + t) * emb_net_size(s1):]
            W0, b0 = p[:s1], p[s1:2 * s1]
            q = p[2 * s1:]
            W1, b1 = q[:s1 * 2 * s1].reshape(s1, 2 * s1), q[s1 * 2 * s1: s1 * 2 * s1 + 2 * s1]
            q = q[s1 * 2 * s1 + 2 * s1:]
            W2, b2 = q[:2 * s1 * 4 * s1].reshape(2 * s1, 4 * s1), q[2 * s1 * 4 * s1: 2 * s1 * 4 * s1 + 4 * s1]
            for x in (-0.8, 0.05, 1.9):
                h0 = np.tanh(x * W0 + b0)
                h1 = np.concatenate([h0, h0]) + np.tanh(h0 @ W1 + b1)
                h2 = np.concatenate([h1, h1]) + np.tanh(h1 @ W2 + b2)
                assert np.allclose(o.embed(a, t, x), h2, rtol=1e-14, atol=1e-15)


def test_fitting_net_pins():
    spec, emb, fit = small_model(ntypes=1, s1=4, m_axis=3, fit_width=8)
    dim, w = spec.dim_descrpt, spec.fit_width
    assert fit.size == fit_net_size(dim, w)
    o = Oracle.from_spec(spec, emb, fit)
    rng = np.random.default_rng(0)
    D = rng.standard_normal(dim)
    W0, p = fit[:dim * w].reshape(dim, w), fit[dim * w:]
    b0, p = p[:w], p[w:]
    W1, p = p[:w * w].reshape(w, w), p[w * w:]
    b1, p = p[:w], p[w:]
    W2, p = p[:w * w].reshape(w, w), p[w * w:]
    b2, p = p[:w], p[w:]
    w3, b3 = p[:w], p[w]
    z0 = np.tanh(D @ W0 + b0)                      # first layer: no skip (reading R4)
    z1 = z0 + np.tanh(z0 @ W1 + b1)                # Eq. 3
    z2 = z1 + np.tanh(z1 @ W2 + b2)
    assert abs(o.fit_net(0, D) - (z2 @ w3 + b3)) < 1e-13
    # zero hidden weights: E = sum_o 3 tanh(b_o)... simplest special case: all zero except b3 -> E = b3
    z = np.zeros_like(fit)
    z[-1] = 1.25
    assert Oracle.from_spec(spec, emb, z).fit_net(0, D) == 1.25


def test_isolated_pair_descriptor_closed_form():
    """Two atoms: T = g (x) (s, s d^) so D[b][a] = 2 s^2 g_b g_a (Eq. 4 with one neighbour); an isolated atom
    has D = 0, E_i = N(0), F = 0."""
    spec, emb, fit = small_model(ntypes=1, s1=4, m_axis=3, fit_width=8, sel=(6,))
    o = Oracle.from_spec(spec, emb, fit)
    box = np.diag([30.0] * 3).reshape(9)
    coord = np.array([[3.0, 4.0, 5.0], [4.2, 5.1, 3.7], [20.0, 20.0, 20.0]])
    types = np.zeros(3, dtype=np.int32)
    nl, _ = o.build_nlist(coord, types, box)
    out = o.atom_rows(coord, types, box, None, nl, want_T=True)
    d = coord[1] - coord[0]
    r = np.linalg.norm(d)
    s = o.switch(r)[0] / r
    g = o.embed(0, 0, s)
    T = np.outer(g, np.concatenate([[s], s * d / r]))
    assert np.allclose(out["T"][0], T, rtol=1e-14, atol=1e-16)
    D = 2 * s * s * np.outer(g, g[:spec.m_axis])
    assert np.allclose(out["D"][0].reshape(spec.m, spec.m_axis), D, rtol=1e-13, atol=1e-16)
    # isolated atom 2
    assert np.all(out["T"][2] == 0) and np.all(out["D"][2] == 0)
    assert out["atom_energy"][2] == o.fit_net(0, np.zeros(spec.dim_descrpt))
    full = o.eval(coord, types, box)
    assert np.all(full["force"][2] == 0)
    assert np.allclose(full["force"][0], -full["force"][1], atol=1e-15)
    # the pair force is along d (central symmetry of a two-body configuration)
    f0 = full["force"][0]
    assert np.linalg.norm(np.cross(f0, d)) < 1e-12 * max(1.0, np.linalg.norm(f0))
    assert abs(full["energy"] - out["atom_energy"].sum()) < 1e-14
