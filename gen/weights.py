"""Random-init network weights in the flat layout of the C ABI (include/dpb.h).

BASELINE.json: "Weights are random-init N(0, 1/fan_in) with biases N(0, 1), all fp64" — variance 1/fan_in,
bias standard deviation 1.  No DP arithmetic here: only draws and array packing.
"""
from __future__ import annotations

from dataclasses import dataclass, field
import numpy as np

from .systems import SEED_BASE


@dataclass(frozen=True)
class ModelSpec:
    name: str
    ntypes: int
    rcut: float
    rcut_smth: float
    sel: tuple
    emb_s1: int                 # embedding widths s1 -> 2 s1 -> 4 s1 = M
    m_axis: int = 16            # M^<
    fit_width: int = 240
    config_id: int = 0

    @property
    def nm(self) -> int:
        return int(sum(self.sel))

    @property
    def m(self) -> int:
        return 4 * self.emb_s1

    @property
    def dim_descrpt(self) -> int:
        return self.m * self.m_axis


WATER = ModelSpec("water", 2, 6.0, 0.5, (46, 92), 25, 16, 240, 0)
COPPER = ModelSpec("copper", 1, 8.0, 2.0, (512,), 32, 16, 240, 2)
# the copper model as the paper states it (PAPER.md:294 embedding 25-50-100, :296 Nm = 500);
# BASELINE.json's copper configs use 32-64-128 and sel 512 (readings R16, R17).
COPPER_PAPER = ModelSpec("copper-paper", 1, 8.0, 2.0, (500,), 25, 16, 240, 2)
MODELS = {"W192": WATER, "W24k": WATER, "Cu32k": COPPER, "Cu864k": COPPER, "Cu32k-paper": COPPER_PAPER}


def emb_net_size(s1: int) -> int:
    """doubles in one embedding net: W0[1][s1] b0[s1] W1[s1][2s1] b1[2s1] W2[2s1][4s1] b2[4s1]."""
    return s1 + s1 + s1 * 2 * s1 + 2 * s1 + 2 * s1 * 4 * s1 + 4 * s1


def fit_net_size(dim_in: int, width: int) -> int:
    """doubles in one fitting net: W0[D][w] b0[w] W1[w][w] b1[w] W2[w][w] b2[w] w3[w] b3[1]."""
    return dim_in * width + width + 2 * (width * width + width) + width + 1


def make_weights(spec: ModelSpec, seed: int | None = None):
    """Return (emb_weights, fit_weights) flat float64 arrays.

    emb_weights holds ntypes*ntypes nets, net (a = centre type, t = neighbour type) at index a*ntypes + t;
    fit_weights holds ntypes nets.  All matrices are row-major [in][out].
    """
    if seed is None:
        seed = SEED_BASE + 100 + spec.config_id
    rng = np.random.default_rng(seed)
    s1 = spec.emb_s1

    def dense(fan_in, fan_out):
        w = rng.standard_normal((fan_in, fan_out)) / np.sqrt(fan_in)
        b = rng.standard_normal(fan_out)
        return [w.reshape(-1), b]

    emb = []
    for _ in range(spec.ntypes * spec.ntypes):
        emb += dense(1, s1) + dense(s1, 2 * s1) + dense(2 * s1, 4 * s1)
    fit = []
    for _ in range(spec.ntypes):
        fit += dense(spec.dim_descrpt, spec.fit_width) + dense(spec.fit_width, spec.fit_width) \
            + dense(spec.fit_width, spec.fit_width) + dense(spec.fit_width, 1)
    emb = np.ascontiguousarray(np.concatenate(emb))
    fit = np.ascontiguousarray(np.concatenate(fit))
    assert emb.size == spec.ntypes ** 2 * emb_net_size(s1)
    assert fit.size == spec.ntypes * fit_net_size(spec.dim_descrpt, spec.fit_width)
    return emb, fit


def condition_fit_w0(spec: ModelSpec, fit: np.ndarray, scale: float | None = None) -> np.ndarray:
    """The 'conditioned' weight set: the first fitting matrix times 1/Nm, so that the first
    fitting layer is not saturated and upstream errors are visible in E and F."""
    if scale is None:
        scale = 1.0 / spec.nm
    out = fit.copy()
    per = fit_net_size(spec.dim_descrpt, spec.fit_width)
    for a in range(spec.ntypes):
        out[a * per: a * per + spec.dim_descrpt * spec.fit_width] *= scale
    return out
