"""Spatial domain decomposition around dpb_eval_local.

One process per GPU; each rank owns the atoms of one brick of an orthorhombic periodic box.  One evaluation is

  1. forward exchange  — every rank receives, as ghost atoms, the atoms of the neighbouring bricks (and the periodic
                         images) within r_c of its brick: three stages (x, y, z), two point-to-point messages each, a
                         later stage forwarding the ghosts of the earlier ones (edges and corners need no diagonal
                         messages);
  2. dpb_eval_local    — E_i of the local atoms, forces on local AND ghost atoms, the local part of the virial;
  3. reverse exchange  — the ghost force increments go back to the owners along the same routes, in reverse order,
                         and are ADDED there (grad_{r_i} E_j != -grad_{r_j} E_i, so they cannot be dropped);
  4. all-reduce        — E and the nine virial components, ten doubles.

Everything here is plumbing.  For CUDA tensors the selection, packing (with the periodic shift) and the force fold-back
are kernels of libdpb (csrc/dd.cu: dpb_dd_pack / dpb_dd_unpack / dpb_dd_add_forces) and the messages travel with
torch.distributed point-to-point calls (NCCL over NVLink); one host synchronisation per stage (the message sizes).  For
CPU tensors (the gloo tests of the routes) the same steps are torch indexing.  All arithmetic of the model runs in the
`evaluate_local` callable — DPModel.eval_local in production; there is no CPU evaluation in this module.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Callable, List, Optional, Sequence, Tuple

import numpy as np


def _torch():
    import torch
    return torch


def choose_grid(world: int, box_lengths: Sequence[float]) -> Tuple[int, int, int]:
    """Factor `world` into px * py * pz with bricks as close to cubes as possible (smallest surface, fewest ghosts)."""
    best, best_cost = (world, 1, 1), None
    L = [float(v) for v in box_lengths]
    for px in range(1, world + 1):
        if world % px:
            continue
        for py in range(1, world // px + 1):
            if (world // px) % py:
                continue
            pz = world // (px * py)
            w = (L[0] / px, L[1] / py, L[2] / pz)
            cost = w[0] * w[1] + w[1] * w[2] + w[0] * w[2]
            if best_cost is None or cost < best_cost - 1e-12:
                best, best_cost = (px, py, pz), cost
    return best


@dataclass
class _Stage:
    """Bookkeeping of one forward stage, kept for the reverse exchange."""
    dim: int
    send_idx: List["object"] = field(default_factory=list)     # [2] index tensors into the atom array (+ then - direction)
    recv_range: List[Tuple[int, int]] = field(default_factory=list)   # [2] slices of the atom array (from - then from +)


class BrickDecomposition:
    """Brick (ix, iy, iz) of a px x py x pz grid over an orthorhombic periodic box; rank = (ix * py + iy) * pz + iz."""

    def __init__(self, box, rcut: float, grid: Optional[Sequence[int]] = None, rank: Optional[int] = None,
                 world: Optional[int] = None, group=None):
        torch = _torch()
        import torch.distributed as dist
        b = np.asarray(box, dtype=np.float64).reshape(3, 3)
        if np.abs(b - np.diag(np.diag(b))).max() != 0.0:
            raise ValueError("box must be orthorhombic")
        self.L = np.diag(b).copy()
        self.rcut = float(rcut)
        self.group = group
        if world is None:
            world = dist.get_world_size(group) if dist.is_available() and dist.is_initialized() else 1
        if rank is None:
            rank = dist.get_rank(group) if dist.is_available() and dist.is_initialized() else 0
        self.world, self.rank = int(world), int(rank)
        self.grid = tuple(int(g) for g in (grid if grid is not None else choose_grid(self.world, self.L)))
        if self.grid[0] * self.grid[1] * self.grid[2] != self.world:
            raise ValueError(f"grid {self.grid} does not match world size {self.world}")
        width = self.L / np.asarray(self.grid)
        if (width < self.rcut).any():
            raise ValueError(f"brick {width} narrower than r_c = {self.rcut}: ghosts would come from beyond the "
                             "nearest neighbour")
        px, py, pz = self.grid
        self.index = (self.rank // (py * pz), (self.rank // pz) % py, self.rank % pz)
        self.lo = width * np.asarray(self.index)
        self.hi = width * (np.asarray(self.index) + 1)
        for c in range(3):
            if self.index[c] == self.grid[c] - 1:
                self.hi[c] = self.L[c]
        self.stages: List[_Stage] = []
        self.nloc = 0
        self._bufs, self._x, self._t = {}, None, None               # device path: reused exchange buffers
        self._torch = torch
        self._dist = dist

    # ---- topology ------------------------------------------------------------------------------------------
    def rank_of(self, index) -> int:
        px, py, pz = self.grid
        return ((index[0] % px) * py + (index[1] % py)) * pz + (index[2] % pz)

    def neighbour(self, dim: int, step: int) -> int:
        idx = list(self.index)
        idx[dim] += step
        return self.rank_of(idx)

    def bounds(self) -> np.ndarray:
        """(lo[3], hi[3]) of the region that holds the local atoms and every ghost: the brick widened by r_c."""
        return np.concatenate([self.lo - self.rcut, self.hi + self.rcut])

    def owned_mask(self, coord):
        """Atoms of a replicated global configuration that this rank owns (wrapped position inside its brick)."""
        torch = self._torch
        L = torch.as_tensor(self.L, dtype=coord.dtype, device=coord.device)
        w = coord - torch.floor(coord / L) * L
        lo = torch.as_tensor(self.lo, dtype=coord.dtype, device=coord.device)
        hi = torch.as_tensor(self.hi, dtype=coord.dtype, device=coord.device)
        return ((w >= lo) & (w < hi)).all(dim=1), w

    # ---- point-to-point plumbing -----------------------------------------------------------------------------
    def _exchange(self, to_plus, to_minus, dim: int):
        """Send `to_plus` to the +dim neighbour and `to_minus` to the -dim neighbour ([k, w] float64 each); returns what
        arrives from the -dim neighbour and from the +dim neighbour.  Neighbour == self: a local copy."""
        torch, dist = self._torch, self._dist
        plus, minus = self.neighbour(dim, +1), self.neighbour(dim, -1)
        if plus == self.rank and minus == self.rank:
            return to_plus.clone(), to_minus.clone()
        dev, w = to_plus.device, to_plus.shape[1]
        n_send = torch.tensor([to_plus.shape[0], to_minus.shape[0]], dtype=torch.int64, device=dev)
        n_from_minus = torch.zeros(1, dtype=torch.int64, device=dev)
        n_from_plus = torch.zeros(1, dtype=torch.int64, device=dev)
        # message order between one pair of ranks is preserved, so with two bricks in this dimension (plus == minus) the
        # first message is the one sent upwards
        # (gloo also matches on the tag: 0 = sent upwards, 1 = sent downwards)
        ops = [dist.P2POp(dist.isend, n_send[0:1], plus, self.group, 0), dist.P2POp(dist.isend, n_send[1:2], minus, self.group, 1),
               dist.P2POp(dist.irecv, n_from_minus, minus, self.group, 0), dist.P2POp(dist.irecv, n_from_plus, plus, self.group, 1)]
        for r in dist.batch_isend_irecv(ops):
            r.wait()
        from_minus = torch.empty((int(n_from_minus.item()), w), dtype=to_plus.dtype, device=dev)
        from_plus = torch.empty((int(n_from_plus.item()), w), dtype=to_plus.dtype, device=dev)
        ops = []
        if to_plus.shape[0]:
            ops.append(dist.P2POp(dist.isend, to_plus.contiguous(), plus, self.group, 0))
        if to_minus.shape[0]:
            ops.append(dist.P2POp(dist.isend, to_minus.contiguous(), minus, self.group, 1))
        if from_minus.shape[0]:
            ops.append(dist.P2POp(dist.irecv, from_minus, minus, self.group, 0))
        if from_plus.shape[0]:
            ops.append(dist.P2POp(dist.irecv, from_plus, plus, self.group, 1))
        if ops:
            for r in dist.batch_isend_irecv(ops):
                r.wait()
        return from_minus, from_plus

    def _exchange_fixed(self, to_plus, to_minus, n_from_minus: int, n_from_plus: int, dim: int):
        """Same routes with sizes both sides already know (reverse exchange)."""
        torch, dist = self._torch, self._dist
        plus, minus = self.neighbour(dim, +1), self.neighbour(dim, -1)
        if plus == self.rank and minus == self.rank:
            return to_plus.clone(), to_minus.clone()
        from_minus = torch.empty((n_from_minus, to_plus.shape[1]), dtype=to_plus.dtype, device=to_plus.device)
        from_plus = torch.empty((n_from_plus, to_plus.shape[1]), dtype=to_plus.dtype, device=to_plus.device)
        ops = []
        if to_plus.shape[0]:
            ops.append(dist.P2POp(dist.isend, to_plus.contiguous(), plus, self.group, 0))
        if to_minus.shape[0]:
            ops.append(dist.P2POp(dist.isend, to_minus.contiguous(), minus, self.group, 1))
        if n_from_minus:
            ops.append(dist.P2POp(dist.irecv, from_minus, minus, self.group, 0))
        if n_from_plus:
            ops.append(dist.P2POp(dist.irecv, from_plus, plus, self.group, 1))
        if ops:
            for r in dist.batch_isend_irecv(ops):
                r.wait()
        return from_minus, from_plus

    # ---- the four steps --------------------------------------------------------------------------------------
    def forward(self, coord, types):
        """Forward exchange.  coord [nloc, 3] float64 (wrapped into the box, inside this brick), types [nloc] int32.
        Returns (coord_all [nall, 3], types_all [nall]) with the local atoms first; remembers the routes."""
        torch = self._torch
        self.nloc = int(coord.shape[0])
        self.stages = []
        if coord.is_cuda:
            return self._forward_cuda(coord, types)
        # CPU tensors (the gloo tests): the same selection, shifts and routes written with torch indexing
        x = coord
        t = types.to(torch.float64)
        for dim in range(3):
            lo, hi, L = float(self.lo[dim]), float(self.hi[dim]), float(self.L[dim])
            xd = x[:, dim]
            idx_plus = torch.nonzero(xd >= hi - self.rcut, as_tuple=False).flatten()
            idx_minus = torch.nonzero(xd < lo + self.rcut, as_tuple=False).flatten()
            pack_plus = torch.cat([x[idx_plus], t[idx_plus, None]], dim=1)
            pack_minus = torch.cat([x[idx_minus], t[idx_minus, None]], dim=1)
            # across the periodic boundary the receiver sees the image: the last brick sends x - L upwards (to brick 0),
            # brick 0 sends x + L downwards
            if self.index[dim] == self.grid[dim] - 1:
                pack_plus[:, dim] -= L
            if self.index[dim] == 0:
                pack_minus[:, dim] += L
            from_minus, from_plus = self._exchange(pack_plus, pack_minus, dim)
            n0 = int(x.shape[0])
            st = _Stage(dim=dim, send_idx=[idx_plus, idx_minus],
                        recv_range=[(n0, n0 + int(from_minus.shape[0])),
                                    (n0 + int(from_minus.shape[0]), n0 + int(from_minus.shape[0]) + int(from_plus.shape[0]))])
            self.stages.append(st)
            x = torch.cat([x, from_minus[:, :3], from_plus[:, :3]], dim=0)
            t = torch.cat([t, from_minus[:, 3], from_plus[:, 3]], dim=0)
        return x.contiguous(), t.to(torch.int32).contiguous()

    def reverse(self, force_all):
        """Reverse exchange: force_all [nall, 3] (local + ghost) -> force [nloc, 3] with every ghost increment added to
        its owner.  Stages in reverse order: what arrives may belong to a ghost of an earlier stage and travels on."""
        if force_all.is_cuda:
            return self._reverse_cuda(force_all)
        f = force_all.clone()
        for st in reversed(self.stages):
            (a0, a1), (b0, b1) = st.recv_range                    # a: came from the - neighbour, b: from the + neighbour
            idx_plus, idx_minus = st.send_idx
            # the ghosts that came from the + neighbour go back up, those from the - neighbour go back down; what comes
            # back from the + neighbour belongs to the atoms sent upwards
            from_minus, from_plus = self._exchange_fixed(f[b0:b1], f[a0:a1], int(idx_minus.shape[0]),
                                                         int(idx_plus.shape[0]), st.dim)
            f = f[:a0]
            if idx_plus.shape[0]:
                f.index_add_(0, idx_plus, from_plus)
            if idx_minus.shape[0]:
                f.index_add_(0, idx_minus, from_minus)
        assert f.shape[0] == self.nloc
        return f

    # ---- device path: selection, packing and the force fold-back are kernels of libdpb (csrc/dd.cu) ------------------
    def _buffers(self, dim: int, cap: int, dev):
        torch = self._torch
        b = self._bufs.get(dim)
        if b is None or b["cap"] < cap:
            b = {"cap": cap,
                 "pack_minus": torch.empty((cap, 4), dtype=torch.float64, device=dev),
                 "pack_plus": torch.empty((cap, 4), dtype=torch.float64, device=dev),
                 "idx_minus": torch.empty(cap, dtype=torch.int32, device=dev),
                 "idx_plus": torch.empty(cap, dtype=torch.int32, device=dev),
                 "counts": torch.zeros(2, dtype=torch.int32, device=dev)}
            self._bufs[dim] = b
        return b

    def _atoms(self, need: int, keep: int, dev):
        """Atom arrays with room for `need` rows; the first `keep` rows survive a reallocation."""
        torch = self._torch
        if self._x is None or self._x.shape[0] < need or self._x.device != dev:
            cap = int(need * 1.25) + 1024
            x = torch.empty((cap, 3), dtype=torch.float64, device=dev)
            t = torch.empty(cap, dtype=torch.int32, device=dev)
            if keep:
                x[:keep] = self._x[:keep]
                t[:keep] = self._t[:keep]
            self._x, self._t = x, t
        return self._x, self._t

    def _forward_cuda(self, coord, types):
        from . import binding
        torch = self._torch
        dev = coord.device
        n = self.nloc
        width = self.hi - self.lo
        grow = float(np.prod(1.0 + 2.0 * self.rcut / width))
        x, t = self._atoms(int(n * grow * 1.1) + 1024, 0, dev)
        x[:n] = coord
        t[:n] = types
        for dim in range(3):
            lo, hi, L = float(self.lo[dim]), float(self.hi[dim]), float(self.L[dim])
            shift_plus = -L if self.index[dim] == self.grid[dim] - 1 else 0.0
            shift_minus = L if self.index[dim] == 0 else 0.0
            cap = min(n, int(n * self.rcut / width[dim] * 1.3) + 256)
            while True:
                b = self._buffers(dim, cap, dev)
                binding.dd_pack(x, t, n, dim, lo + self.rcut, hi - self.rcut, shift_minus, shift_plus, b["pack_minus"],
                                b["idx_minus"], b["pack_plus"], b["idx_plus"], b["counts"])
                km, kp = (int(v) for v in b["counts"].tolist())          # the one host synchronisation of the stage
                if max(km, kp) <= b["cap"]:
                    break
                cap = max(km, kp)
            to_plus, to_minus = b["pack_plus"][:kp], b["pack_minus"][:km]
            if self.neighbour(dim, +1) == self.rank and self.neighbour(dim, -1) == self.rank:
                from_minus, from_plus = to_plus, to_minus                 # the images of this brick's own atoms
            else:
                from_minus, from_plus = self._exchange(to_plus, to_minus, dim)
            k0, k1 = int(from_minus.shape[0]), int(from_plus.shape[0])
            x, t = self._atoms(n + k0 + k1, n, dev)
            binding.dd_unpack(from_minus, k0, x[n:], t[n:])
            binding.dd_unpack(from_plus, k1, x[n + k0:], t[n + k0:])
            self.stages.append(_Stage(dim=dim, send_idx=[b["idx_plus"][:kp], b["idx_minus"][:km]],
                                      recv_range=[(n, n + k0), (n + k0, n + k0 + k1)]))
            n += k0 + k1
        return x[:n], t[:n]

    def _reverse_cuda(self, f):
        """In place on the evaluator's force array (local + ghost rows); returns the view of the local rows."""
        from . import binding
        for st in reversed(self.stages):
            (a0, a1), (b0, b1) = st.recv_range
            idx_plus, idx_minus = st.send_idx
            if self.neighbour(st.dim, +1) == self.rank and self.neighbour(st.dim, -1) == self.rank:
                from_minus, from_plus = f[b0:b1], f[a0:a1]                # ghost rows lie behind every target row
            else:
                from_minus, from_plus = self._exchange_fixed(f[b0:b1], f[a0:a1], int(idx_minus.shape[0]),
                                                             int(idx_plus.shape[0]), st.dim)
            binding.dd_add_forces(idx_plus, from_plus, int(idx_plus.shape[0]), f)
            binding.dd_add_forces(idx_minus, from_minus, int(idx_minus.shape[0]), f)
        return f[:self.nloc]

    def evaluate(self, evaluate_local: Callable, coord, types):
        """One evaluation of the decomposed system.  `evaluate_local(coord_all, types_all, nloc, bounds)` must return a
        dict with energy [1], atom_energy [nloc], force [nall, 3], virial [3, 3] (DPModel.eval_local).  Returns
        dict(energy (global, on every rank), virial (global), force [nloc, 3], atom_energy [nloc], nall)."""
        torch, dist = self._torch, self._dist
        x, t = self.forward(coord, types)
        out = evaluate_local(x, t, self.nloc, self.bounds())
        force = self.reverse(out["force"])
        red = torch.cat([out["energy"].reshape(1), out["virial"].reshape(9)]).contiguous()
        if self.world > 1:
            dist.all_reduce(red, op=dist.ReduceOp.SUM, group=self.group)
        return {"energy": red[0:1], "virial": red[1:].reshape(3, 3), "force": force,
                "atom_energy": out["atom_energy"], "nall": int(x.shape[0])}

    # ---- molecular dynamics on the decomposition: atom migration and the time loop -----------------------------------
    def migrate(self, coord, vel, types, tags=None):
        """Atoms that left the brick move to the neighbour that now owns them (three stages, as the ghost exchange; an
        atom may move less than one brick width per call).  Rows of (x, v, type, tag) travel together; the periodic shift
        is applied by the sender, so local coordinates always lie inside [lo, hi).  `tags` (optional, one number per atom,
        e.g. a global index below 2^53) travels with its atom.  Returns the new (coord, vel, types, tags)."""
        torch = self._torch
        x, v, t = coord, vel, types.to(torch.float64)
        g = (tags if tags is not None else torch.zeros(x.shape[0], device=x.device)).to(torch.float64)
        for dim in range(3):
            lo, hi, L = float(self.lo[dim]), float(self.hi[dim]), float(self.L[dim])
            up, dn = x[:, dim] >= hi, x[:, dim] < lo
            iu, idn = torch.nonzero(up).flatten(), torch.nonzero(dn).flatten()
            pack_up = torch.cat([x[iu], v[iu], t[iu, None], g[iu, None]], dim=1)
            pack_dn = torch.cat([x[idn], v[idn], t[idn, None], g[idn, None]], dim=1)
            if self.index[dim] == self.grid[dim] - 1:
                pack_up[:, dim] -= L
            if self.index[dim] == 0:
                pack_dn[:, dim] += L
            from_minus, from_plus = self._exchange(pack_up, pack_dn, dim)
            keep = torch.nonzero(~(up | dn)).flatten()
            x = torch.cat([x[keep], from_minus[:, 0:3], from_plus[:, 0:3]], dim=0)
            v = torch.cat([v[keep], from_minus[:, 3:6], from_plus[:, 3:6]], dim=0)
            t = torch.cat([t[keep], from_minus[:, 6], from_plus[:, 6]], dim=0)
            g = torch.cat([g[keep], from_minus[:, 7], from_plus[:, 7]], dim=0)
        return x.contiguous(), v.contiguous(), t.to(torch.int32).contiguous(), (g if tags is not None else None)

    def md_run(self, evaluate_local: Callable, integrator, coord, vel, types, nsteps: int, thermo_every: int = 1,
               tags=None):
        """Velocity-Verlet NVE on the decomposed system: per step kick + drift, migration, ghost exchange,
        dpb_eval_local, reverse exchange, kick.  `integrator` supplies kick_drift / kick / kinetic_energy
        (binding.CudaIntegrator: libdpb's kernels).  Returns (coord, vel, types, tags) of this rank's atoms after the
        run and thermo [k][2] = global (E_pot, E_kin) at steps 0, thermo_every, ..."""
        torch, dist = self._torch, self._dist
        thermo = []

        def record(out):
            ek = integrator.kinetic_energy(vel, types).reshape(1).to(torch.float64)
            if self.world > 1:
                dist.all_reduce(ek, op=dist.ReduceOp.SUM, group=self.group)
            thermo.append(torch.cat([out["energy"].reshape(1), ek]))

        coord, vel, types, tags = self.migrate(coord, vel, types, tags)
        out = self.evaluate(evaluate_local, coord, types)
        force = out["force"].contiguous()
        record(out)
        for step in range(1, nsteps + 1):
            integrator.kick_drift(coord, vel, force, types)
            coord, vel, types, tags = self.migrate(coord, vel, types, tags)
            out = self.evaluate(evaluate_local, coord, types)
            force = out["force"].contiguous()
            integrator.kick(vel, force, types)
            if step % thermo_every == 0:
                record(out)
        return coord, vel, types, tags, torch.stack(thermo)
