"""Synthetic periodic boxes standing in for the paper's workloads (§4).

The paper's equilibrated 192-atom water cell and its trained models are not available, so positions are built
from a seed with the density, species mix, cutoff and neighbour counts of the paper's systems (BASELINE.json
`configs`).  Nothing here computes any part of the DP model.
"""
from __future__ import annotations

from dataclasses import dataclass
import numpy as np

SEED_BASE = 200411658          # arXiv number of the paper; config k uses SEED_BASE + k for positions


@dataclass(frozen=True)
class SystemSpec:
    name: str
    kind: str                  # "water" | "copper"
    cells: int                 # water: grid edge (sites per dim); copper: FCC unit cells per dim
    bcc: bool                  # water only: body-centred grid (2 sites per cell)
    box_len: float             # cubic box edge, Angstrom
    jitter: float              # Gaussian sigma per Cartesian component, Angstrom
    config_id: int             # index into BASELINE.json `configs`


# BASELINE.json `configs` 0..4 (config 3 = config 1's inputs in mixed precision).
CONFIGS = {
    "W192":   SystemSpec("W192",   "water",  4,  False, 12.42, 0.10, 0),
    "W24k":   SystemSpec("W24k",   "water",  16, True,  62.1,  0.10, 1),
    "Cu32k":  SystemSpec("Cu32k",  "copper", 20, False, 20 * 3.634, 0.05, 2),
    "Cu864k": SystemSpec("Cu864k", "copper", 60, False, 60 * 3.634, 0.05, 4),
    # same box as Cu32k; the model is the paper's own copper model (gen.weights.COPPER_PAPER), SURVEY.md §8(f) NEXT #4
    "Cu32k-paper": SystemSpec("Cu32k-paper", "copper", 20, False, 20 * 3.634, 0.05, 2),
}

_OH = 0.96                      # O-H bond length, Angstrom
_HOH = np.deg2rad(104.5)        # H-O-H angle


def _random_rotations(rng: np.random.Generator, n: int) -> np.ndarray:
    """n uniform random rotation matrices from normalised 4-Gaussian quaternions."""
    q = rng.standard_normal((n, 4))
    q /= np.linalg.norm(q, axis=1, keepdims=True)
    w, x, y, z = q[:, 0], q[:, 1], q[:, 2], q[:, 3]
    rot = np.empty((n, 3, 3))
    rot[:, 0, 0] = 1 - 2 * (y * y + z * z); rot[:, 0, 1] = 2 * (x * y - z * w); rot[:, 0, 2] = 2 * (x * z + y * w)
    rot[:, 1, 0] = 2 * (x * y + z * w); rot[:, 1, 1] = 1 - 2 * (x * x + z * z); rot[:, 1, 2] = 2 * (y * z - x * w)
    rot[:, 2, 0] = 2 * (x * z - y * w); rot[:, 2, 1] = 2 * (y * z + x * w); rot[:, 2, 2] = 1 - 2 * (x * x + y * y)
    return rot


def water_box(grid: int, bcc: bool, box_len: float, jitter: float, seed: int):
    """Water molecules on a simple-cubic (or body-centred) grid with random orientation and Gaussian jitter.

    Returns (coord [N,3] float64 wrapped into [0,L), type [N] int32 with O=0/H=1 in O,H,H order, box [9]).
    """
    rng = np.random.default_rng(seed)
    a = box_len / grid
    idx = np.stack(np.meshgrid(np.arange(grid), np.arange(grid), np.arange(grid), indexing="ij"), -1).reshape(-1, 3)
    sites = (idx + 0.5) * a
    if bcc:
        sites = np.concatenate([sites, (idx + 1.0) * a], axis=0)
    nmol = sites.shape[0]
    half = 0.5 * _HOH
    h_local = np.array([[+_OH * np.sin(half), 0.0, _OH * np.cos(half)],
                        [-_OH * np.sin(half), 0.0, _OH * np.cos(half)]])
    rot = _random_rotations(rng, nmol)
    coord = np.empty((nmol, 3, 3))
    coord[:, 0, :] = sites
    coord[:, 1, :] = sites + np.einsum("nab,b->na", rot, h_local[0])
    coord[:, 2, :] = sites + np.einsum("nab,b->na", rot, h_local[1])
    coord = coord.reshape(-1, 3)
    coord += rng.normal(0.0, jitter, size=coord.shape)
    coord = np.mod(coord, box_len)
    coord[coord >= box_len] = 0.0      # np.mod may return L for tiny negative inputs
    types = np.tile(np.array([0, 1, 1], dtype=np.int32), nmol)
    box = np.diag([box_len] * 3).reshape(9).astype(np.float64)
    return np.ascontiguousarray(coord), types, box


def copper_box(cells: int, jitter: float, seed: int, a: float = 3.634):
    """FCC copper (lattice constant PAPER.md:298) with thermal jitter; single species."""
    rng = np.random.default_rng(seed)
    basis = np.array([[0.0, 0.0, 0.0], [0.5, 0.5, 0.0], [0.5, 0.0, 0.5], [0.0, 0.5, 0.5]])
    idx = np.stack(np.meshgrid(np.arange(cells), np.arange(cells), np.arange(cells), indexing="ij"), -1).reshape(-1, 1, 3)
    coord = ((idx + basis[None, :, :]) * a).reshape(-1, 3)
    box_len = cells * a
    if jitter > 0.0:
        coord = coord + rng.normal(0.0, jitter, size=coord.shape)
    coord = np.mod(coord, box_len)
    coord[coord >= box_len] = 0.0
    types = np.zeros(coord.shape[0], dtype=np.int32)
    box = np.diag([box_len] * 3).reshape(9).astype(np.float64)
    return np.ascontiguousarray(coord), types, box


def make_system(name: str, seed: int | None = None):
    """Build one of the BASELINE.json configurations by name ("W192", "W24k", "Cu32k", "Cu864k")."""
    spec = CONFIGS[name]
    if seed is None:
        seed = SEED_BASE + spec.config_id
    if spec.kind == "water":
        return water_box(spec.cells, spec.bcc, spec.box_len, spec.jitter, seed)
    return copper_box(spec.cells, spec.jitter, seed)


def perturbed(coord: np.ndarray, box: np.ndarray, sigma: float, seed: int) -> np.ndarray:
    """Fresh Gaussian perturbation of the base positions (config 1: sigma = 0.01 A between calls), wrapped."""
    rng = np.random.default_rng(seed)
    L = np.array([box[0], box[4], box[8]])
    out = np.mod(coord + rng.normal(0.0, sigma, size=coord.shape), L)
    out = np.where(out >= L, 0.0, out)
    return np.ascontiguousarray(out)


def replicate(coord: np.ndarray, types: np.ndarray, box: np.ndarray, reps: int):
    """reps x reps x reps periodic replication (used by the extensivity pin)."""
    L = np.array([box[0], box[4], box[8]])
    shifts = np.stack(np.meshgrid(np.arange(reps), np.arange(reps), np.arange(reps), indexing="ij"), -1).reshape(-1, 3)
    big = (coord[None, :, :] + shifts[:, None, :] * L).reshape(-1, 3)
    return np.ascontiguousarray(big), np.tile(types, shifts.shape[0]).astype(np.int32), np.diag(L * reps).reshape(9)


# ---- molecular dynamics inputs (330 K) ------------------------------------
MASSES = {"W192": (15.999, 1.008), "W24k": (15.999, 1.008), "Cu32k": (63.546,), "Cu864k": (63.546,),
          "Cu32k-paper": (63.546,)}   # amu

# CODATA 2018: atomic mass constant, elementary charge, Boltzmann constant
_AMU_KG, _E_C, _KB_J = 1.66053906660e-27, 1.602176634e-19, 1.380649e-23
AMU_A2_FS2_IN_EV = _AMU_KG * 1e10 / _E_C            # 1 amu A^2 / fs^2 in eV (103.6427)
KB_EV = _KB_J / _E_C                                # eV / K


def maxwell_boltzmann(types: np.ndarray, masses, temperature: float, seed: int) -> np.ndarray:
    """Velocities [N][3] in A/fs drawn from the Maxwell-Boltzmann distribution at `temperature` (K), with the total
    momentum removed and then rescaled so that 2 E_kin / (3 N k_B) equals `temperature` exactly."""
    rng = np.random.default_rng(seed)
    m = np.asarray(masses, dtype=np.float64)[np.asarray(types)]
    sigma = np.sqrt(KB_EV * temperature / (m * AMU_A2_FS2_IN_EV))
    v = rng.standard_normal((len(m), 3)) * sigma[:, None]
    v -= (m[:, None] * v).sum(0) / m.sum()
    ek = 0.5 * (m[:, None] * v * v).sum() * AMU_A2_FS2_IN_EV
    v *= np.sqrt(1.5 * len(m) * KB_EV * temperature / ek)
    return np.ascontiguousarray(v)
