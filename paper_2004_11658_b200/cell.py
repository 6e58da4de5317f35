"""General (triclinic) periodic cells through explicit images.

dpb_eval takes an orthorhombic box with r_c < L/2.  Any other periodic cell — triclinic, or thinner than 2 r_c — is
evaluated the way the paper formulates periodicity: the atoms of the cell are the local atoms, their lattice images
within r_c of the cell are ghost atoms, dpb_eval_local does the arithmetic, and the ghost forces are added back to the
atoms they are images of.  This module only builds the images and folds the forces (torch indexing on the device the
coordinates live on); every step of the model runs in dpb_eval_local.
"""
from __future__ import annotations

import itertools

import numpy as np


def _torch():
    import torch
    return torch


def cell_heights(cell) -> np.ndarray:
    """Perpendicular heights h_c = V / |a_j x a_k| of the parallelepiped spanned by the rows of `cell`."""
    a = np.asarray(cell, dtype=np.float64).reshape(3, 3)
    vol = abs(np.linalg.det(a))
    if not vol > 0.0:
        raise ValueError("cell is singular")
    return np.array([vol / np.linalg.norm(np.cross(a[(c + 1) % 3], a[(c + 2) % 3])) for c in range(3)])


def periodic_images(coord, cell, rcut: float):
    """coord [N, 3] (torch, any device) in a cell whose rows are the lattice vectors.  Returns
    (coord_all [nall, 3] with the N wrapped atoms first, owner [nall] int64 index of the atom each row is an image of,
    bounds (lo[3], hi[3]) numpy).  An image is kept when its fractional coordinate s_c lies in
    [-r_c / h_c, 1 + r_c / h_c] for every c: a superset of the atoms within r_c of the cell."""
    torch = _torch()
    a = np.asarray(cell, dtype=np.float64).reshape(3, 3)
    h = cell_heights(a)
    A = torch.as_tensor(a, dtype=torch.float64, device=coord.device)
    Ainv = torch.as_tensor(np.linalg.inv(a), dtype=torch.float64, device=coord.device)
    s = coord @ Ainv                                           # fractional coordinates: x = s A
    s = s - torch.floor(s)
    margin = torch.as_tensor(rcut / h, dtype=torch.float64, device=coord.device)
    n = [int(np.ceil(rcut / hc)) for hc in h]                   # image shells per lattice direction
    parts, owners = [s], [torch.arange(coord.shape[0], device=coord.device)]
    for shift in itertools.product(*(range(-k, k + 1) for k in n)):
        if shift == (0, 0, 0):
            continue
        t = s + torch.as_tensor(shift, dtype=torch.float64, device=coord.device)
        keep = ((t >= -margin) & (t <= 1.0 + margin)).all(dim=1)
        idx = torch.nonzero(keep).flatten()
        if idx.numel():
            parts.append(t[idx])
            owners.append(idx)
    x = torch.cat(parts) @ A
    owner = torch.cat(owners)
    # bounding box of the widened parallelepiped: its 8 corners in fractional coordinates
    m = rcut / h
    corners = np.array([[(-m[c] if (k >> c) & 1 == 0 else 1.0 + m[c]) for c in range(3)] for k in range(8)]) @ a
    pad = 1e-9 * (1.0 + np.abs(corners).max())
    return x.contiguous(), owner, (corners.min(axis=0) - pad, corners.max(axis=0) + pad)


def eval_cell(model, coord, types, cell):
    """Energy, forces, virial and E_i of N atoms in a general periodic cell (rows = lattice vectors; triclinic allowed,
    r_c may exceed half the cell).  `model` is a DPModel; coord [N, 3] float64 and types [N] int32 are CUDA tensors."""
    torch = _torch()
    n = int(coord.shape[0])
    x, owner, (lo, hi) = periodic_images(coord, cell, model.rcut)
    out = model.eval_local(x, types[owner].contiguous(), n, np.concatenate([lo, hi]))
    force = torch.zeros((n, 3), dtype=torch.float64, device=coord.device)
    force.index_add_(0, owner, out["force"])                    # ghost increments go to the atoms they are images of
    return {"energy": out["energy"], "atom_energy": out["atom_energy"], "force": force, "virial": out["virial"],
            "nall": int(x.shape[0])}
