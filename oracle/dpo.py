"""ctypes binding of oracle/libdpo.so (argument marshalling only; all arithmetic is in dpo.c).

TEST INFRASTRUCTURE — see oracle/dpo.h for who may use it.
"""
from __future__ import annotations

import ctypes as C

import numpy as np

from . import build as _build


class _Desc(C.Structure):
    _fields_ = [("ntypes", C.c_int32), ("rcut", C.c_double), ("rcut_smth", C.c_double),
                ("sel", C.POINTER(C.c_int32)), ("emb_s1", C.c_int32), ("m_axis", C.c_int32),
                ("fit_width", C.c_int32), ("emb_weights", C.POINTER(C.c_double)),
                ("fit_weights", C.POINTER(C.c_double))]


_dp = C.POINTER(C.c_double)
_ip = C.POINTER(C.c_int32)
_lp = C.POINTER(C.c_int64)


def _d(a):
    return None if a is None else a.ctypes.data_as(_dp)


def _i(a):
    return None if a is None else a.ctypes.data_as(_ip)


def _l(a):
    return None if a is None else a.ctypes.data_as(_lp)


class OracleError(RuntimeError):
    pass


class Oracle:
    """One DP model (host weights) bound to libdpo.so."""

    def __init__(self, ntypes, rcut, rcut_smth, sel, emb_s1, m_axis, fit_width, emb_weights, fit_weights):
        self.lib = C.CDLL(_build.build())
        self.lib.dpo_fit.restype = C.c_double
        self.ntypes, self.rcut, self.rcut_smth = int(ntypes), float(rcut), float(rcut_smth)
        self.sel = np.ascontiguousarray(sel, dtype=np.int32)
        self.s1, self.m_axis, self.fit_width = int(emb_s1), int(m_axis), int(fit_width)
        self.emb = np.ascontiguousarray(emb_weights, dtype=np.float64)
        self.fit = np.ascontiguousarray(fit_weights, dtype=np.float64)
        self.nm = int(self.sel.sum())
        self.M = 4 * self.s1
        self.dim = self.M * self.m_axis
        self.desc = _Desc(self.ntypes, self.rcut, self.rcut_smth, _i(self.sel), self.s1, self.m_axis,
                          self.fit_width, _d(self.emb), _d(self.fit))

    @classmethod
    def from_spec(cls, spec, emb, fit):
        return cls(spec.ntypes, spec.rcut, spec.rcut_smth, spec.sel, spec.emb_s1, spec.m_axis, spec.fit_width,
                   emb, fit)

    @staticmethod
    def _chk(rc, what):
        if rc != 0:
            raise OracleError(f"{what} failed with status {rc}")

    def num_threads(self) -> int:
        return int(self.lib.dpo_num_threads())

    def switch(self, r):
        w, dw = C.c_double(), C.c_double()
        self.lib.dpo_switch(C.c_double(r), C.c_double(self.rcut_smth), C.c_double(self.rcut), C.byref(w),
                            C.byref(dw))
        return w.value, dw.value

    def displacement(self, ri, rj, L):
        ri, rj, L = (np.ascontiguousarray(a, dtype=np.float64) for a in (ri, rj, L))
        d, r = np.zeros(3), C.c_double()
        self.lib.dpo_displacement(_d(ri), _d(rj), _d(L), _d(d), C.byref(r))
        return d, r.value

    @staticmethod
    def _inputs(coord, types, box):
        coord = np.ascontiguousarray(coord, dtype=np.float64).reshape(-1, 3)
        types = np.ascontiguousarray(types, dtype=np.int32)
        box = np.ascontiguousarray(box, dtype=np.float64).reshape(9)
        return coord, types, box

    def build_nlist(self, coord, types, box, rows=None, cells=False):
        """Formatted neighbour list; returns (nlist [nrows][Nm] int32, n_overflow)."""
        coord, types, box = self._inputs(coord, types, box)
        n = coord.shape[0]
        ovf = C.c_int64(0)
        if cells:
            assert rows is None
            nlist = np.empty((n, self.nm), dtype=np.int32)
            rc = self.lib.dpo_build_nlist_cells(C.byref(self.desc), C.c_int64(n), _d(coord), _i(types), _d(box),
                                                _i(nlist), C.byref(ovf))
        else:
            rows_a = None if rows is None else np.ascontiguousarray(rows, dtype=np.int64)
            nrows = n if rows is None else rows_a.size
            nlist = np.empty((nrows, self.nm), dtype=np.int32)
            rc = self.lib.dpo_build_nlist_rows(C.byref(self.desc), C.c_int64(n), _d(coord), _i(types), _d(box),
                                               C.c_int64(nrows), _l(rows_a), _i(nlist), C.byref(ovf))
        self._chk(rc, "dpo_build_nlist")
        return nlist, int(ovf.value)

    def env_row(self, coord, types, box, i, nlist_row):
        coord, types, box = self._inputs(coord, types, box)
        row = np.ascontiguousarray(nlist_row, dtype=np.int32)
        env, denv, disp = np.empty((self.nm, 4)), np.empty((self.nm, 4, 3)), np.empty((self.nm, 3))
        rc = self.lib.dpo_env_row(C.byref(self.desc), C.c_int64(coord.shape[0]), _d(coord), _d(box),
                                  C.c_int64(i), _i(row), _d(env), _d(denv), _d(disp))
        self._chk(rc, "dpo_env_row")
        return env, denv, disp

    def net_offset(self, a, t):
        s1 = self.s1
        return (a * self.ntypes + t) * (2 * s1 + s1 * 2 * s1 + 2 * s1 + 2 * s1 * 4 * s1 + 4 * s1)

    def embed(self, a, t, x):
        g = np.empty(self.M)
        off = self.net_offset(a, t)
        self.lib.dpo_embed(_d(self.emb[off:]), C.c_int32(self.s1), C.c_double(x), _d(g))
        return g

    def fit_net(self, a, D):
        D = np.ascontiguousarray(D, dtype=np.float64)
        w = self.fit_width
        per = self.dim * w + w + 2 * (w * w + w) + w + 1
        return float(self.lib.dpo_fit(_d(self.fit[a * per:]), C.c_int32(self.dim), C.c_int32(w), _d(D)))

    def atom_rows(self, coord, types, box, rows, nlist_rows, want_T=False):
        """E_i and dE_i/dd_ik for the listed atoms.  Returns dict(atom_energy, fslot[, T, D, dT])."""
        coord, types, box = self._inputs(coord, types, box)
        rows_a = None if rows is None else np.ascontiguousarray(rows, dtype=np.int64)
        nrows = coord.shape[0] if rows is None else rows_a.size
        nl = np.ascontiguousarray(nlist_rows, dtype=np.int32).reshape(nrows, self.nm)
        ei = np.empty(nrows)
        fs = np.empty((nrows, self.nm, 3))
        T = np.empty((nrows, self.M, 4)) if want_T else None
        D = np.empty((nrows, self.dim)) if want_T else None
        dT = np.empty((nrows, self.M, 4)) if want_T else None
        rc = self.lib.dpo_atom_rows(C.byref(self.desc), C.c_int64(coord.shape[0]), _d(coord), _i(types), _d(box),
                                    C.c_int64(nrows), _l(rows_a), _i(nl), _d(ei), _d(fs), _d(T), _d(D), _d(dT))
        self._chk(rc, "dpo_atom_rows")
        out = {"atom_energy": ei, "fslot": fs}
        if want_T:
            out.update(T=T, D=D, dT=dT)
        return out

    def eval(self, coord, types, box, cells=False, want_nlist=True):
        """One full evaluation.  Returns dict(energy, atom_energy, force, virial[, nlist])."""
        coord, types, box = self._inputs(coord, types, box)
        n = coord.shape[0]
        e = C.c_double(0.0)
        ei, f, vir = np.empty(n), np.empty((n, 3)), np.empty(9)
        nlist = np.empty((n, self.nm), dtype=np.int32) if want_nlist else None
        rc = self.lib.dpo_eval(C.byref(self.desc), C.c_int64(n), _d(coord), _i(types), _d(box), C.byref(e),
                               _d(ei), _d(f), _d(vir), _i(nlist), C.c_int(1 if cells else 0))
        self._chk(rc, "dpo_eval")
        out = {"energy": e.value, "atom_energy": ei, "force": f, "virial": vir.reshape(3, 3)}
        if want_nlist:
            out["nlist"] = nlist
        return out

    def atom_virial(self, coord, types, box):
        """Per-atom virial [N, 3, 3], centre-atom split (dpo_atom_virial)."""
        coord, types, box = self._inputs(coord, types, box)
        n = coord.shape[0]
        out = np.empty((max(n, 1), 9))
        rc = self.lib.dpo_atom_virial(C.byref(self.desc), C.c_int64(n), _d(coord), _i(types), _d(box), _d(out))
        self._chk(rc, "dpo_atom_virial")
        return out[:n].reshape(n, 3, 3)

    def eval_local(self, coord, types, nloc, want_nlist=True):
        """One sub-region with explicit ghost atoms, no box (dpo_eval_local): atoms [0, nloc) are
        local.  Returns dict(energy, atom_energy[nloc], force[nall], virial[, nlist[nloc]])."""
        coord = np.ascontiguousarray(coord, dtype=np.float64).reshape(-1, 3)
        types = np.ascontiguousarray(types, dtype=np.int32)
        nall = coord.shape[0]
        e = C.c_double(0.0)
        ei, f, vir = np.empty(max(nloc, 1)), np.empty((nall, 3)), np.empty(9)
        nlist = np.empty((max(nloc, 1), self.nm), dtype=np.int32) if want_nlist else None
        rc = self.lib.dpo_eval_local(C.byref(self.desc), C.c_int64(nloc), C.c_int64(nall), _d(coord), _i(types),
                                     C.byref(e), _d(ei), _d(f), _d(vir), _i(nlist))
        self._chk(rc, "dpo_eval_local")
        out = {"energy": e.value, "atom_energy": ei[:nloc], "force": f, "virial": vir.reshape(3, 3)}
        if want_nlist:
            out["nlist"] = nlist[:nloc]
        return out

    def md_run(self, coord, vel, types, mass, box, dt_fs, nsteps, thermo_every=1, cells=False):
        """Velocity-Verlet NVE MD (dpo_md_run).  Returns (coord, vel, thermo[k][4] = (E_pot, E_kin, T, P [bar]))."""
        coord, types, box = self._inputs(coord, types, box)
        coord = coord.copy()
        vel = np.ascontiguousarray(vel, dtype=np.float64).reshape(-1, 3).copy()
        mass = np.ascontiguousarray(mass, dtype=np.float64)
        nt = nsteps // thermo_every + 1
        thermo = np.zeros((nt, 4))
        rc = self.lib.dpo_md_run(C.byref(self.desc), C.c_int64(coord.shape[0]), _d(coord), _d(vel), _i(types),
                                 _d(mass), _d(box), C.c_double(dt_fs), C.c_int64(nsteps), C.c_int64(thermo_every),
                                 _d(thermo), C.c_int(1 if cells else 0))
        self._chk(rc, "dpo_md_run")
        return coord, vel, thermo
