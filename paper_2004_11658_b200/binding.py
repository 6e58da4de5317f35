"""ctypes binding of libdpb.so — same names as include/dpb.h, argument marshalling only."""
from __future__ import annotations

import ctypes as C
import os
from dataclasses import dataclass

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))

STATUS = {0: "DPB_OK", -1: "DPB_EINVAL", -2: "DPB_EBOX", -3: "DPB_ENOMEM", -4: "DPB_ECUDA", -5: "DPB_ECAP",
          -6: "DPB_ENOTIMPL"}
FP64, TF32, BF16, BF16_PLAIN = 0, 1, 2, 3


class DPBError(RuntimeError):
    def __init__(self, status: int, message: str):
        super().__init__(f"{STATUS.get(status, status)}: {message}")
        self.status = status


class _Desc(C.Structure):
    _fields_ = [("ntypes", C.c_int32), ("rcut", C.c_double), ("rcut_smth", C.c_double),
                ("sel", C.POINTER(C.c_int32)), ("emb_s1", C.c_int32), ("m_axis", C.c_int32),
                ("fit_width", C.c_int32), ("emb_weights", C.POINTER(C.c_double)),
                ("fit_weights", C.POINTER(C.c_double))]


class _MDParams(C.Structure):
    _fields_ = [("dt_fs", C.c_double), ("nsteps", C.c_int32), ("thermo_every", C.c_int32),
                ("rebuild_every", C.c_int32), ("reserved", C.c_int32), ("skin", C.c_double)]


class _MDInfo(C.Structure):
    _fields_ = [("n_thermo", C.c_int32), ("n_rebuilds", C.c_int32), ("skin_violated", C.c_int32),
                ("reserved", C.c_int32), ("max_displacement", C.c_double)]


class _Info(C.Structure):
    _fields_ = [("n_real_pairs", C.c_int64), ("n_overflow", C.c_int64), ("max_nei", C.c_int32 * 8),
                ("n_chunks", C.c_int32), ("reserved", C.c_int32)]


@dataclass
class EvalInfo:
    n_real_pairs: int
    n_overflow: int
    max_nei: tuple
    n_chunks: int


def lib_path() -> str:
    """The in-tree build (paper_2004_11658_b200/build.py); there is no other place the library is looked for."""
    return os.path.join(HERE, "libdpb.so")


_LIB = None


def load_library():
    """Load libdpb.so (built in-tree by paper_2004_11658_b200/build.py).  Raises if it is missing: no fallback."""
    global _LIB
    if _LIB is not None:
        return _LIB
    path = lib_path()
    if not os.path.exists(path):
        raise DPBError(-4, f"{path} not found: build it with `python -m paper_2004_11658_b200.build` "
                           "(there is no CPU fallback)")
    lib = C.CDLL(path)
    vp, i64, i32 = C.c_void_p, C.c_int64, C.c_int
    lib.dpb_model_create.argtypes = [C.POINTER(_Desc), i32, C.POINTER(vp)]
    lib.dpb_model_destroy.argtypes = [vp]
    lib.dpb_model_nm.argtypes = [vp]
    lib.dpb_model_set_chunk.argtypes = [vp, i64]
    lib.dpb_model_set_variant.argtypes = [vp, i32]
    lib.dpb_model_set_deterministic.argtypes = [vp, i32]
    lib.dpb_model_set_pair_reuse.argtypes = [vp, i32]
    lib.dpb_model_set_stored_activations.argtypes = [vp, i32]
    lib.dpb_model_set_species_pipeline.argtypes = [vp, i32]
    lib.dpb_model_set_atom_virial.argtypes = [vp, vp]
    lib.dpb_model_set_timing.argtypes = [vp, i32]
    lib.dpb_model_stage_us.argtypes = [vp, C.POINTER(C.c_float)]
    lib.dpb_set_debug_buffers.argtypes = [vp, vp, vp, vp]
    lib.dpb_debug_sorted_order.argtypes = [vp, vp, i64, vp]
    lib.dpb_model_status.argtypes = [vp, vp]
    lib.dpb_model_set_graph.argtypes = [vp, i32]
    lib.dpb_eval.argtypes = [vp, vp, i64, vp, vp, C.POINTER(C.c_double), vp, vp, vp, vp, vp, C.POINTER(_Info)]
    lib.dpb_eval_local.argtypes = [vp, vp, i64, i64, vp, vp, C.POINTER(C.c_double), vp, vp, vp, vp, vp,
                                   C.POINTER(_Info)]
    lib.dpb_eval_host.argtypes = lib.dpb_eval.argtypes
    lib.dpb_eval_cell.argtypes = [vp, vp, i64, vp, vp, C.POINTER(C.c_double), vp, vp, vp, vp, C.POINTER(_Info)]
    lib.dpb_build_nlist.argtypes = [vp, vp, i64, vp, vp, C.POINTER(C.c_double), vp, C.POINTER(i64)]
    lib.dpb_build_nlist_static.argtypes = [vp, vp, i64, vp, vp, C.POINTER(C.c_double), vp, vp]
    lib.dpb_md_run.argtypes = [vp, vp, i64, vp, vp, vp, C.POINTER(C.c_double), C.POINTER(C.c_double),
                               C.POINTER(_MDParams), vp, C.POINTER(_MDInfo)]
    d = C.c_double
    lib.dpb_dd_pack.argtypes = [vp, i64, vp, vp, i32, d, d, d, d, i64, vp, vp, vp, vp, vp]
    lib.dpb_dd_unpack.argtypes = [vp, i64, vp, vp, vp]
    lib.dpb_md_coefficients.argtypes = [C.POINTER(C.c_double), i32, d, C.POINTER(C.c_double)]
    lib.dpb_md_kick_drift.argtypes = [vp, i64, vp, vp, vp, vp, vp, d]
    lib.dpb_md_kick.argtypes = [vp, i64, vp, vp, vp, vp]
    lib.dpb_md_kinetic_energy.argtypes = [vp, i64, vp, vp, vp, vp]
    lib.dpb_dd_add_forces.argtypes = [vp, i64, vp, vp, vp]
    lib.dpb_kernel_launches.restype = C.c_int64
    lib.dpb_last_error.restype = C.c_char_p
    lib.dpb_version.restype = C.c_char_p
    _LIB = lib
    return lib


def _torch():
    import torch
    return torch


class DPModel:
    """One DP model on the current CUDA device (dpb_model_create / dpb_eval / dpb_model_destroy)."""

    def __init__(self, ntypes, rcut, rcut_smth, sel, emb_s1, m_axis, fit_width, emb_weights, fit_weights,
                 precision: int = FP64):
        self.lib = load_library()
        torch = _torch()
        if not torch.cuda.is_available():
            raise DPBError(-4, "no CUDA device: this library has no CPU path")
        self.ntypes = int(ntypes)
        self.sel = np.ascontiguousarray(sel, dtype=np.int32)
        self.nm = int(self.sel.sum())
        self.rcut, self.rcut_smth = float(rcut), float(rcut_smth)
        self.s1, self.m_axis, self.fit_width = int(emb_s1), int(m_axis), int(fit_width)
        self.M = 4 * self.s1
        self.dim = self.M * self.m_axis
        emb = np.ascontiguousarray(emb_weights, dtype=np.float64)
        fit = np.ascontiguousarray(fit_weights, dtype=np.float64)
        desc = _Desc(self.ntypes, float(rcut), float(rcut_smth), self.sel.ctypes.data_as(C.POINTER(C.c_int32)),
                     self.s1, self.m_axis, self.fit_width, emb.ctypes.data_as(C.POINTER(C.c_double)),
                     fit.ctypes.data_as(C.POINTER(C.c_double)))
        self._h = C.c_void_p()
        self._chk(self.lib.dpb_model_create(C.byref(desc), int(precision), C.byref(self._h)))

    @classmethod
    def from_spec(cls, spec, emb, fit, precision: int = FP64):
        return cls(spec.ntypes, spec.rcut, spec.rcut_smth, spec.sel, spec.emb_s1, spec.m_axis, spec.fit_width,
                   emb, fit, precision)

    def _chk(self, rc):
        if rc != 0:
            raise DPBError(rc, self.lib.dpb_last_error().decode())

    def close(self):
        if getattr(self, "_h", None) is not None and self._h:
            self.lib.dpb_model_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_chunk(self, n: int):
        self._chk(self.lib.dpb_model_set_chunk(self._h, int(n)))

    def set_variant(self, v: int):
        self._chk(self.lib.dpb_model_set_variant(self._h, int(v)))

    def set_deterministic(self, on: bool):
        self._chk(self.lib.dpb_model_set_deterministic(self._h, int(bool(on))))

    def set_species_pipeline(self, on: bool):
        """dpb_model_set_species_pipeline: the stages of one centre type back to back on its stream (default on)."""
        self._chk(self.lib.dpb_model_set_species_pipeline(self._h, int(bool(on))))

    def set_stored_activations(self, on: bool):
        """dpb_model_set_stored_activations: pass 2 reads the embedding activations pass 1 stored (default on)."""
        self._chk(self.lib.dpb_model_set_stored_activations(self._h, int(bool(on))))

    def set_pair_reuse(self, on: int):
        """dpb_model_set_pair_reuse: 0 off, 1 single-chunk evaluations (default), 2 always."""
        self._chk(self.lib.dpb_model_set_pair_reuse(self._h, int(on)))

    def set_graph(self, mode: int):
        """dpb_model_set_graph: 0 off, 1 evaluations of at most 4096 atoms (default), 2 always."""
        self._chk(self.lib.dpb_model_set_graph(self._h, int(mode)))

    def set_atom_virial(self, buf=None):
        """dpb_model_set_atom_virial: a CUDA float64 [N, 9] (or [N, 3, 3]) tensor that the following evaluations fill with
        the per-atom virial (needs set_deterministic(True)); None switches it off.  The tensor is kept alive here."""
        if buf is not None:
            torch = _torch()
            assert buf.is_cuda and buf.dtype == torch.float64 and buf.is_contiguous()
        self._atom_virial_keep = buf
        self._chk(self.lib.dpb_model_set_atom_virial(self._h, None if buf is None else C.c_void_p(buf.data_ptr())))

    def set_timing(self, on: bool):
        self._chk(self.lib.dpb_model_set_timing(self._h, int(bool(on))))

    def stage_us(self):
        buf = (C.c_float * 8)()
        self._chk(self.lib.dpb_model_stage_us(self._h, buf))
        return list(buf)

    def kernel_launches(self) -> int:
        return int(self.lib.dpb_kernel_launches())

    def set_debug_buffers(self, T=None, D=None, dT=None):
        p = [None if t is None else C.c_void_p(t.data_ptr()) for t in (T, D, dT)]
        self._debug_keep = (T, D, dT)
        self._chk(self.lib.dpb_set_debug_buffers(self._h, *p))

    def status(self):
        """dpb_model_status: synchronise and raise DPBError if the last evaluation hit a deferred input error."""
        self._chk(self.lib.dpb_model_status(self._h, self._stream()))

    def sorted_order(self, natoms: int):
        """dpb_debug_sorted_order: CUDA int32 [natoms], input index of the atom at every sorted position of the last call."""
        torch = _torch()
        order = torch.empty(int(natoms), dtype=torch.int32, device="cuda")
        self._chk(self.lib.dpb_debug_sorted_order(self._h, self._stream(), int(natoms), C.c_void_p(order.data_ptr())))
        return order

    @staticmethod
    def _box(box):
        b = np.ascontiguousarray(box, dtype=np.float64).reshape(9)
        return b, b.ctypes.data_as(C.POINTER(C.c_double))

    @staticmethod
    def _stream():
        torch = _torch()
        return C.c_void_p(torch.cuda.current_stream().cuda_stream)

    def eval(self, coord, types, box, want_nlist=False, want_info=False, out=None):
        """dpb_eval on torch CUDA tensors (coord float64 [N,3], types int32 [N]); returns a dict of CUDA tensors.

        `out` may hold preallocated tensors (energy, atom_energy, force, virial, nlist) to reuse between calls.
        """
        torch = _torch()
        assert coord.is_cuda and coord.dtype == torch.float64 and coord.is_contiguous()
        assert types.is_cuda and types.dtype == torch.int32 and types.is_contiguous()
        n = int(coord.shape[0])
        dev = coord.device
        o = out if out is not None else {}
        if "energy" not in o:
            o["energy"] = torch.empty(1, dtype=torch.float64, device=dev)
            o["atom_energy"] = torch.empty(n, dtype=torch.float64, device=dev)
            o["force"] = torch.empty((n, 3), dtype=torch.float64, device=dev)
            o["virial"] = torch.empty((3, 3), dtype=torch.float64, device=dev)
        if want_nlist and "nlist" not in o:
            o["nlist"] = torch.empty((n, self.nm), dtype=torch.int32, device=dev)
        b, bp = self._box(box)
        info = _Info() if want_info else None
        nl = C.c_void_p(o["nlist"].data_ptr()) if want_nlist else None
        rc = self.lib.dpb_eval(self._h, self._stream(), n, C.c_void_p(coord.data_ptr()), C.c_void_p(types.data_ptr()),
                               bp, C.c_void_p(o["energy"].data_ptr()), C.c_void_p(o["atom_energy"].data_ptr()),
                               C.c_void_p(o["force"].data_ptr()), C.c_void_p(o["virial"].data_ptr()), nl,
                               C.byref(info) if want_info else None)
        self._chk(rc)
        if want_info:
            o["info"] = EvalInfo(int(info.n_real_pairs), int(info.n_overflow), tuple(info.max_nei), int(info.n_chunks))
        return o

    def eval_local(self, coord, types, nloc, bounds, want_nlist=False, want_info=True):
        """dpb_eval_local: atoms [0, nloc) local, the rest ghosts; bounds = (lo[3], hi[3]) containing all of them."""
        torch = _torch()
        assert coord.is_cuda and coord.dtype == torch.float64 and coord.is_contiguous()
        assert types.is_cuda and types.dtype == torch.int32 and types.is_contiguous()
        nall = int(coord.shape[0])
        dev = coord.device
        o = {"energy": torch.empty(1, dtype=torch.float64, device=dev),
             "atom_energy": torch.empty(max(nloc, 1), dtype=torch.float64, device=dev)[:nloc],
             "force": torch.empty((max(nall, 1), 3), dtype=torch.float64, device=dev)[:nall],
             "virial": torch.empty((3, 3), dtype=torch.float64, device=dev)}
        if want_nlist:
            o["nlist"] = torch.empty((max(nloc, 1), self.nm), dtype=torch.int32, device=dev)[:nloc]
        bnd = (C.c_double * 6)(*[float(v) for v in np.asarray(bounds, dtype=np.float64).reshape(-1)])
        info = _Info() if want_info else None
        rc = self.lib.dpb_eval_local(self._h, self._stream(), C.c_int64(nloc), C.c_int64(nall),
                                     C.c_void_p(coord.data_ptr()), C.c_void_p(types.data_ptr()), bnd,
                                     C.c_void_p(o["energy"].data_ptr()), C.c_void_p(o["atom_energy"].data_ptr()),
                                     C.c_void_p(o["force"].data_ptr()), C.c_void_p(o["virial"].data_ptr()),
                                     C.c_void_p(o["nlist"].data_ptr()) if want_nlist else None,
                                     C.byref(info) if want_info else None)
        self._chk(rc)
        if want_info:
            o["info"] = EvalInfo(int(info.n_real_pairs), int(info.n_overflow), tuple(info.max_nei), int(info.n_chunks))
        return o

    def eval_cell(self, coord, types, cell, want_info=False):
        """dpb_eval_cell: N atoms in a general periodic cell (rows of `cell` = lattice vectors; triclinic allowed, r_c may
        exceed half the cell).  coord float64 [N,3] and types int32 [N] are CUDA tensors; returns a dict of CUDA tensors."""
        torch = _torch()
        assert coord.is_cuda and coord.dtype == torch.float64 and coord.is_contiguous()
        assert types.is_cuda and types.dtype == torch.int32 and types.is_contiguous()
        n = int(coord.shape[0])
        dev = coord.device
        o = {"energy": torch.empty(1, dtype=torch.float64, device=dev),
             "atom_energy": torch.empty(max(n, 1), dtype=torch.float64, device=dev)[:n],
             "force": torch.empty((max(n, 1), 3), dtype=torch.float64, device=dev)[:n],
             "virial": torch.empty((3, 3), dtype=torch.float64, device=dev)}
        b, bp = self._box(cell)
        info = _Info() if want_info else None
        rc = self.lib.dpb_eval_cell(self._h, self._stream(), n, C.c_void_p(coord.data_ptr()), C.c_void_p(types.data_ptr()),
                                    bp, C.c_void_p(o["energy"].data_ptr()), C.c_void_p(o["atom_energy"].data_ptr()),
                                    C.c_void_p(o["force"].data_ptr()), C.c_void_p(o["virial"].data_ptr()),
                                    C.byref(info) if want_info else None)
        self._chk(rc)
        if want_info:
            o["info"] = EvalInfo(int(info.n_real_pairs), int(info.n_overflow), tuple(info.max_nei), int(info.n_chunks))
        return o

    def eval_host(self, coord, types, box, out=None, want_nlist=False):
        """dpb_eval_host on HOST arrays (numpy or pinned torch CPU tensors): H2D, evaluation, D2H, synchronise."""
        torch = _torch()

        def ptr(a):
            return C.c_void_p(a.data_ptr()) if isinstance(a, torch.Tensor) else C.c_void_p(a.ctypes.data)

        n = int(coord.shape[0])
        o = out if out is not None else {}
        if "energy" not in o:
            o["energy"] = np.empty(1)
            o["atom_energy"] = np.empty(n)
            o["force"] = np.empty((n, 3))
            o["virial"] = np.empty((3, 3))
        if want_nlist and "nlist" not in o:
            o["nlist"] = np.empty((n, self.nm), dtype=np.int32)
        b, bp = self._box(box)
        rc = self.lib.dpb_eval_host(self._h, self._stream(), n, ptr(coord), ptr(types), bp, ptr(o["energy"]),
                                    ptr(o["atom_energy"]), ptr(o["force"]), ptr(o["virial"]),
                                    ptr(o["nlist"]) if want_nlist else None, None)
        self._chk(rc)
        return o

    def build_nlist(self, coord, types, box):
        """dpb_build_nlist: returns (nlist CUDA int32 [N][Nm], n_overflow)."""
        torch = _torch()
        n = int(coord.shape[0])
        nlist = torch.empty((n, self.nm), dtype=torch.int32, device=coord.device)
        b, bp = self._box(box)
        ovf = C.c_int64(0)
        rc = self.lib.dpb_build_nlist(self._h, self._stream(), n, C.c_void_p(coord.data_ptr()),
                                      C.c_void_p(types.data_ptr()), bp, C.c_void_p(nlist.data_ptr()), C.byref(ovf))
        self._chk(rc)
        return nlist, int(ovf.value)

    def build_nlist_static(self, coord, types, box, nlist, status=None):
        """dpb_build_nlist_static: Alg. 1 with no allocation (scratch in a fixed device array; at most 4096 atoms and
        natoms * Nm <= 262144).  nlist (CUDA int32 [N][Nm]) and status (CUDA int64 [4] or None) are the caller's."""
        torch = _torch()
        n = int(coord.shape[0])
        assert nlist.is_cuda and nlist.dtype == torch.int32 and nlist.is_contiguous() and nlist.numel() >= n * self.nm
        assert status is None or (status.is_cuda and status.dtype == torch.int64 and status.numel() >= 4)
        b, bp = self._box(box)
        rc = self.lib.dpb_build_nlist_static(self._h, self._stream(), n, C.c_void_p(coord.data_ptr()),
                                             C.c_void_p(types.data_ptr()), bp, C.c_void_p(nlist.data_ptr()),
                                             C.c_void_p(status.data_ptr()) if status is not None else None)
        self._chk(rc)
        return nlist

    def md_run(self, coord, vel, types, mass, box, dt_fs, nsteps, thermo_every=1, rebuild_every=1, skin=0.0):
        """dpb_md_run: velocity-Verlet NVE on torch CUDA tensors coord / vel (float64 [N,3], updated IN PLACE).
        Returns (thermo numpy [k][4] = (E_pot, E_kin, T, P [bar]), info dict)."""
        torch = _torch()
        assert coord.is_cuda and coord.dtype == torch.float64 and coord.is_contiguous()
        assert vel.is_cuda and vel.dtype == torch.float64 and vel.is_contiguous()
        assert types.is_cuda and types.dtype == torch.int32 and types.is_contiguous()
        n = int(coord.shape[0])
        b, bp = self._box(box)
        m = np.ascontiguousarray(mass, dtype=np.float64)
        prm = _MDParams(float(dt_fs), int(nsteps), int(thermo_every), int(rebuild_every), 0, float(skin))
        thermo = np.zeros((nsteps // thermo_every + 1, 4))
        info = _MDInfo()
        rc = self.lib.dpb_md_run(self._h, self._stream(), n, C.c_void_p(coord.data_ptr()), C.c_void_p(vel.data_ptr()),
                                 C.c_void_p(types.data_ptr()), m.ctypes.data_as(C.POINTER(C.c_double)), bp,
                                 C.byref(prm), C.c_void_p(thermo.ctypes.data), C.byref(info))
        self._chk(rc)
        return thermo, dict(n_thermo=info.n_thermo, n_rebuilds=info.n_rebuilds, skin_violated=bool(info.skin_violated),
                            max_displacement=info.max_displacement)


# ---- ghost exchange kernels of the domain decomposition (dd.py); argument marshalling only ----------------------
def _dd_chk(lib, rc):
    if rc != 0:
        raise DPBError(rc, lib.dpb_last_error().decode())


def dd_pack(coord, types, n, dim, cut_minus, cut_plus, shift_minus, shift_plus, pack_minus, idx_minus, pack_plus,
            idx_plus, counts):
    """dpb_dd_pack on torch CUDA tensors: atoms [0, n) of coord / types; capacity = rows of the pack buffers."""
    lib = load_library()
    p = lambda t: C.c_void_p(t.data_ptr())
    cap = int(pack_minus.shape[0])
    assert int(pack_plus.shape[0]) == cap and int(idx_minus.shape[0]) >= cap and int(idx_plus.shape[0]) >= cap
    _dd_chk(lib, lib.dpb_dd_pack(DPModel._stream(), n, p(coord), p(types), dim, cut_minus, cut_plus, shift_minus,
                                 shift_plus, cap, p(pack_minus), p(idx_minus), p(pack_plus), p(idx_plus), p(counts)))


def dd_unpack(pack, k, coord_out, type_out):
    lib = load_library()
    p = lambda t: C.c_void_p(t.data_ptr())
    _dd_chk(lib, lib.dpb_dd_unpack(DPModel._stream(), k, p(pack), p(coord_out), p(type_out)))


def dd_add_forces(idx, fin, k, force):
    lib = load_library()
    p = lambda t: C.c_void_p(t.data_ptr())
    _dd_chk(lib, lib.dpb_dd_add_forces(DPModel._stream(), k, p(idx), p(fin), p(force)))


# ---- velocity-Verlet pieces (dpb_md_*): the integrator of the decomposition's MD driver -----------------------------
class CudaIntegrator:
    """Kick / drift / kinetic energy on CUDA tensors through libdpb's kernels (csrc/md.cu)."""

    def __init__(self, masses, dt_fs: float, device):
        torch = _torch()
        self.lib = load_library()
        m = np.ascontiguousarray(masses, dtype=np.float64)
        self.ntypes, self.dt = int(m.size), float(dt_fs)
        co = np.zeros(2 * self.ntypes)
        _dd_chk(self.lib, self.lib.dpb_md_coefficients(m.ctypes.data_as(C.POINTER(C.c_double)), self.ntypes, self.dt,
                                                      co.ctypes.data_as(C.POINTER(C.c_double))))
        self.coeff = torch.tensor(co, device=device)
        self._ek = torch.zeros(1, dtype=torch.float64, device=device)

    def kick_drift(self, coord, vel, force, types):
        p = lambda t: C.c_void_p(t.data_ptr())
        assert coord.is_contiguous() and vel.is_contiguous() and force.is_contiguous()
        _dd_chk(self.lib, self.lib.dpb_md_kick_drift(DPModel._stream(), int(coord.shape[0]), p(coord), p(vel), p(force),
                                                    p(types), p(self.coeff), self.dt))

    def kick(self, vel, force, types):
        p = lambda t: C.c_void_p(t.data_ptr())
        assert vel.is_contiguous() and force.is_contiguous()
        _dd_chk(self.lib, self.lib.dpb_md_kick(DPModel._stream(), int(vel.shape[0]), p(vel), p(force), p(types),
                                              p(self.coeff)))

    def kinetic_energy(self, vel, types):
        p = lambda t: C.c_void_p(t.data_ptr())
        _dd_chk(self.lib, self.lib.dpb_md_kinetic_energy(DPModel._stream(), int(vel.shape[0]), p(vel), p(types),
                                                        C.c_void_p(self.coeff.data_ptr() + 8 * self.ntypes), p(self._ek)))
        return self._ek.clone()
