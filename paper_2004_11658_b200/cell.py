"""General (triclinic) periodic cells — argument marshalling only.

dpb_eval takes an orthorhombic box with r_c < L/2.  Any other periodic cell — triclinic, or thinner than 2 r_c — goes
through dpb_eval_cell (include/dpb.h): the library wraps the atoms into the cell, builds their lattice images within r_c
of it as ghost atoms, runs dpb_eval_local's kernels and adds the ghost forces back to the atoms they are images of
(csrc/cell.cu).  Nothing is computed here.
"""
from __future__ import annotations


def eval_cell(model, coord, types, cell, want_info=False):
    """Energy, forces, virial and E_i of N atoms in a general periodic cell (rows = lattice vectors; triclinic allowed,
    r_c may exceed half the cell).  `model` is a DPModel; coord [N, 3] float64 and types [N] int32 are CUDA tensors."""
    return model.eval_cell(coord, types, cell, want_info=want_info)
