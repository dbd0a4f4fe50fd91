"""Thin ctypes binding over the C ABI of ``include/md_b200.h`` (argument marshalling only).

Same names as the C entry points.  Buffers may be numpy arrays (host) or torch
tensors (host or CUDA); torch supplies device memory and the stream.  Importing
this module loads ``libmd_b200.so`` and fails loudly if it is missing: there is
no CPU fallback and nothing here ever touches ``oracle/``.
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libmd_b200.so")

MD_OK = 0
MD_ERR_BAD_ARGUMENT, MD_ERR_BOX_TOO_SMALL, MD_ERR_CUDA, MD_ERR_OVERFLOW, MD_ERR_NOT_READY, MD_ERR_NONFINITE = -1, -2, -3, -4, -5, -6
MD_FP64, MD_MIXED = 0, 1
MD_PAIR_LJ126, MD_PAIR_EAM_FS, MD_PAIR_BUCK_COUL, MD_PAIR_EAM_TAB = 1, 2, 3, 4
MD_LIST_FULL, MD_LIST_HALF = 0, 1
MD_THERMO_NONE, MD_THERMO_NOSE_HOOVER = 0, 1
MD_NOALLOC_SCRATCH_BYTES, MD_NOALLOC_MAX_ATOMS = 524288, 16769024
MD_KERNEL_AUTO, MD_KERNEL_TPA, MD_KERNEL_SUBWARP, MD_KERNEL_WARP, MD_KERNEL_CELL, MD_KERNEL_SUBWARP4, MD_KERNEL_SUBWARP2 = 0, 1, 2, 3, 4, 5, 6
KERNEL_NAMES = {0: "auto", 1: "tpa", 2: "subwarp8", 3: "warp", 4: "cell", 5: "subwarp4", 6: "subwarp2"}

EXPORTS = [
    "md_create", "md_destroy", "md_set_units", "md_set_precision", "md_set_positions", "md_set_velocities",
    "md_set_pair", "md_set_neighbor", "md_build_neighbors", "md_compute_forces", "md_run", "md_get_positions",
    "md_get_velocities", "md_get_forces", "md_get_neighbors", "md_get_neighbor_rows", "md_kinetic_energy", "md_autotune",
    "md_get_stats", "md_last_error", "md_set_option", "md_set_pair_coeff", "md_set_type_charges", "md_set_thermostat", "md_get_thermostat", "md_set_eam_tables",
    "md_kinetic_energy_noalloc",
]


class md_stats(ctypes.Structure):
    _fields_ = [
        ("natoms", ctypes.c_int64), ("nsteps_total", ctypes.c_int64), ("nbuilds", ctypes.c_int64),
        ("nforce_evals", ctypes.c_int64), ("kernel_variant", ctypes.c_int32), ("list_kind", ctypes.c_int32),
        ("precision", ctypes.c_int32), ("lanes_per_atom", ctypes.c_int32), ("ncells", ctypes.c_int32 * 3),
        ("brick", ctypes.c_int32 * 3), ("ntiles", ctypes.c_int32), ("tile_capacity", ctypes.c_int32),
        ("max_tile_atoms", ctypes.c_int32), ("max_neighbors", ctypes.c_int32), ("row_capacity", ctypes.c_int32),
        ("list_balanced", ctypes.c_int32), ("mean_neighbors", ctypes.c_double), ("kinetic_energy", ctypes.c_double),
        ("ms_build", ctypes.c_double), ("ms_force", ctypes.c_double), ("ms_run", ctypes.c_double),
        ("launches_last_run", ctypes.c_int64), ("launches_total", ctypes.c_int64),
        ("ms_force_sampled", ctypes.c_double), ("nforce_sampled", ctypes.c_int64),
        ("ms_build_in_run", ctypes.c_double), ("nbuilds_in_run", ctypes.c_int64),
        ("max_row", ctypes.c_int32), ("reserved0", ctypes.c_int32), ("mean_row", ctypes.c_double),
        ("ms_force_pass1_sampled", ctypes.c_double),
    ]

    def as_dict(self) -> dict:
        out = {}
        for name, _ in self._fields_:
            val = getattr(self, name)
            out[name] = list(val) if hasattr(val, "__len__") else val
        return out


class MDError(RuntimeError):
    def __init__(self, code: int, text: str):
        super().__init__("md_b200 error %d: %s" % (code, text))
        self.code = code


def _load():
    if not os.path.exists(LIB_PATH):
        raise ImportError(
            "libmd_b200.so is missing (%s). Build it with `python -m paper_1009_4330_b200.build`; "
            "there is no CPU fallback." % LIB_PATH)
    L = ctypes.CDLL(LIB_PATH)
    vp, dp, ip = ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p   # raw addresses: host or device
    L.md_create.argtypes = [ctypes.POINTER(vp), ctypes.POINTER(ctypes.c_double), ctypes.c_int64, ip, ctypes.c_int,
                            ctypes.POINTER(ctypes.c_double), vp]
    L.md_destroy.argtypes = [vp]
    L.md_destroy.restype = None
    L.md_set_units.argtypes = [vp, ctypes.c_double, ctypes.c_double]
    L.md_set_precision.argtypes = [vp, ctypes.c_int]
    L.md_set_positions.argtypes = [vp, dp]
    L.md_set_velocities.argtypes = [vp, dp]
    L.md_set_pair.argtypes = [vp, ctypes.c_int, ctypes.POINTER(ctypes.c_double), ctypes.c_int, ctypes.c_double,
                              ctypes.c_double]
    L.md_set_neighbor.argtypes = [vp, ctypes.c_int, ctypes.c_int]
    L.md_build_neighbors.argtypes = [vp]
    L.md_compute_forces.argtypes = [vp, dp, ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_double)]
    L.md_run.argtypes = [vp, ctypes.c_int64, ctypes.c_double]
    L.md_get_positions.argtypes = [vp, dp]
    L.md_get_velocities.argtypes = [vp, dp]
    L.md_get_forces.argtypes = [vp, dp]
    L.md_get_neighbors.argtypes = [vp, ip, ip, ctypes.c_int64]
    L.md_get_neighbor_rows.argtypes = [vp, ip, ip, ip, ctypes.c_int64]
    L.md_kinetic_energy.argtypes = [vp, ctypes.POINTER(ctypes.c_double)]
    L.md_set_option.argtypes = [vp, ctypes.c_char_p, ctypes.c_int64]
    L.md_set_eam_tables.argtypes = [vp, ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_double), ctypes.c_int,
                                    ctypes.POINTER(ctypes.c_double), ctypes.c_int]
    L.md_set_thermostat.argtypes = [vp, ctypes.c_int, ctypes.c_double, ctypes.c_double]
    L.md_get_thermostat.argtypes = [vp, ctypes.POINTER(ctypes.c_double)]
    L.md_set_pair_coeff.argtypes = [vp, ctypes.c_int, ctypes.c_int, ctypes.POINTER(ctypes.c_double), ctypes.c_int]
    L.md_set_type_charges.argtypes = [vp, ctypes.POINTER(ctypes.c_double), ctypes.c_int]
    L.md_kinetic_energy_noalloc.argtypes = [dp, ip, dp, ctypes.c_int64, ctypes.c_double, dp, vp]
    L.md_autotune.argtypes = [vp, ctypes.c_int, ctypes.POINTER(ctypes.c_double)]
    L.md_get_stats.argtypes = [vp, ctypes.POINTER(md_stats)]
    L.md_last_error.argtypes = [vp]
    L.md_last_error.restype = ctypes.c_char_p
    for name in EXPORTS:
        if name not in ("md_destroy", "md_last_error"):
            getattr(L, name).restype = ctypes.c_int
    return L


lib = _load()


def _addr(buf, dtype, count):
    """Address of a contiguous numpy array or torch tensor with ``count`` elements of ``dtype``."""
    if isinstance(buf, np.ndarray):
        if buf.dtype != dtype or not buf.flags["C_CONTIGUOUS"] or buf.size != count:
            raise ValueError("expected a C-contiguous %s array with %d elements" % (np.dtype(dtype).name, count))
        return buf.ctypes.data
    if hasattr(buf, "data_ptr"):   # torch tensor
        import torch
        want = {np.dtype(np.float64): torch.float64, np.dtype(np.int32): torch.int32}[np.dtype(dtype)]
        if buf.dtype != want or not buf.is_contiguous() or buf.numel() != count:
            raise ValueError("expected a contiguous %s tensor with %d elements" % (want, count))
        return buf.data_ptr()
    raise TypeError("buffer must be a numpy array or a torch tensor")


def current_stream_ptr() -> int:
    """The current torch CUDA stream as a raw cudaStream_t."""
    import torch
    return int(torch.cuda.current_stream().cuda_stream)


def md_kinetic_energy_noalloc(v, types, mass, mvv2e: float, ke_out, stream: int | None = None):
    """``md_kinetic_energy_noalloc`` of the C ABI: all four buffers are CUDA tensors the caller owns (v: N x 3 float64,
    types: N int32, mass: ntypes float64, ke_out: 1 float64); nothing is allocated and the stream is not synchronised."""
    for t in (v, types, mass, ke_out):
        if not (hasattr(t, "is_cuda") and t.is_cuda):
            raise TypeError("md_kinetic_energy_noalloc takes CUDA tensors")
    n = int(types.numel())
    if stream is None:
        stream = current_stream_ptr()
    rc = lib.md_kinetic_energy_noalloc(_addr(v, np.float64, 3 * n), _addr(types, np.int32, n), _addr(mass, np.float64, mass.numel()),
                                       n, float(mvv2e), _addr(ke_out, np.float64, 1), ctypes.c_void_p(stream))
    if rc != MD_OK:
        raise MDError(rc, (lib.md_last_error(None) or b"").decode())


class System:
    """Owns one ``md_system`` handle.  Methods mirror the C entry points one to one."""

    def __init__(self, box, natoms: int, types, mass, stream: int | None = None):
        box = np.ascontiguousarray(box, dtype=np.float64)
        mass = np.ascontiguousarray(mass, dtype=np.float64)
        self.natoms = int(natoms)
        self._h = ctypes.c_void_p()
        if stream is None:
            stream = current_stream_ptr()
        rc = lib.md_create(ctypes.byref(self._h), box.ctypes.data_as(ctypes.POINTER(ctypes.c_double)), self.natoms,
                           _addr(types, np.int32, self.natoms), len(mass),
                           mass.ctypes.data_as(ctypes.POINTER(ctypes.c_double)), ctypes.c_void_p(stream))
        if rc != MD_OK:
            self._h = ctypes.c_void_p()
            raise MDError(rc, (lib.md_last_error(None) or b"").decode())

    # -- plumbing ---------------------------------------------------------------------------------------
    def _ck(self, rc: int):
        if rc != MD_OK:
            raise MDError(rc, (lib.md_last_error(self._h) or b"").decode())

    def close(self):
        if getattr(self, "_h", None) and self._h.value:
            lib.md_destroy(self._h)
            self._h = ctypes.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- the C entry points -----------------------------------------------------------------------------
    def md_set_units(self, ftm2v: float, mvv2e: float):
        self._ck(lib.md_set_units(self._h, ftm2v, mvv2e))

    def md_set_precision(self, mode: int):
        self._ck(lib.md_set_precision(self._h, mode))

    def md_set_positions(self, x):
        self._ck(lib.md_set_positions(self._h, _addr(x, np.float64, 3 * self.natoms)))

    def md_set_velocities(self, v):
        self._ck(lib.md_set_velocities(self._h, _addr(v, np.float64, 3 * self.natoms)))

    def md_set_pair(self, style: int, params, rc: float, skin: float):
        p = (ctypes.c_double * len(params))(*[float(q) for q in params])
        self._ck(lib.md_set_pair(self._h, style, p, len(params), rc, skin))

    def md_set_pair_coeff(self, type_a: int, type_b: int, coeff):
        c = (ctypes.c_double * len(coeff))(*[float(q) for q in coeff])
        self._ck(lib.md_set_pair_coeff(self._h, int(type_a), int(type_b), c, len(coeff)))

    def md_set_type_charges(self, q):
        c = (ctypes.c_double * len(q))(*[float(v) for v in q])
        self._ck(lib.md_set_type_charges(self._h, c, len(q)))

    def md_set_thermostat(self, kind: int, kT: float = 0.0, tau: float = 0.0):
        self._ck(lib.md_set_thermostat(self._h, int(kind), float(kT), float(tau)))

    def md_get_thermostat(self):
        out = (ctypes.c_double * 3)()
        self._ck(lib.md_get_thermostat(self._h, out))
        return {"xi": out[0], "eta": out[1], "energy": out[2]}

    def md_set_eam_tables(self, rho_r, phi_r, F_rho):
        dp = ctypes.POINTER(ctypes.c_double)
        a, b, c = (np.ascontiguousarray(t, dtype=np.float64) for t in (rho_r, phi_r, F_rho))
        if len(a) != len(b):
            raise ValueError("rho_r and phi_r must have the same length")
        self._ck(lib.md_set_eam_tables(self._h, a.ctypes.data_as(dp), b.ctypes.data_as(dp), len(a), c.ctypes.data_as(dp), len(c)))

    def md_set_neighbor(self, list_kind: int, kernel: int):
        self._ck(lib.md_set_neighbor(self._h, list_kind, kernel))

    def md_build_neighbors(self):
        self._ck(lib.md_build_neighbors(self._h))

    def md_compute_forces(self, f_out=None, energy: bool = False, virial: bool = False):
        """Returns (energy or None, virial[6] or None); fills f_out when given."""
        e = ctypes.c_double(0.0)
        w = (ctypes.c_double * 6)()
        self._ck(lib.md_compute_forces(self._h, _addr(f_out, np.float64, 3 * self.natoms) if f_out is not None else None,
                                       ctypes.byref(e) if energy else None, w if virial else None))
        return (e.value if energy else None), (np.array(list(w)) if virial else None)

    def md_run(self, nsteps: int, dt: float):
        self._ck(lib.md_run(self._h, int(nsteps), float(dt)))

    def md_get_positions(self, x):
        self._ck(lib.md_get_positions(self._h, _addr(x, np.float64, 3 * self.natoms)))

    def md_get_velocities(self, v):
        self._ck(lib.md_get_velocities(self._h, _addr(v, np.float64, 3 * self.natoms)))

    def md_get_forces(self, f):
        self._ck(lib.md_get_forces(self._h, _addr(f, np.float64, 3 * self.natoms)))

    def md_get_neighbors(self, numneigh, neigh, stride: int):
        self._ck(lib.md_get_neighbors(self._h, _addr(numneigh, np.int32, self.natoms),
                                      _addr(neigh, np.int32, self.natoms * stride), stride))

    def md_get_neighbor_rows(self, row_owner, numrow, entries, stride: int):
        self._ck(lib.md_get_neighbor_rows(self._h, _addr(row_owner, np.int32, self.natoms), _addr(numrow, np.int32, self.natoms),
                                          _addr(entries, np.int32, self.natoms * stride), stride))

    def md_set_option(self, name: str, value: int):
        self._ck(lib.md_set_option(self._h, name.encode(), int(value)))

    def md_kinetic_energy(self) -> float:
        ke = ctypes.c_double(0.0)
        self._ck(lib.md_kinetic_energy(self._h, ctypes.byref(ke)))
        return ke.value

    def md_autotune(self, nrep: int = 3):
        ms = (ctypes.c_double * 5)()
        self._ck(lib.md_autotune(self._h, nrep, ms))
        return {"tpa": ms[0], "subwarp8": ms[1], "warp": ms[2], "subwarp4": ms[3], "subwarp2": ms[4]}

    def md_get_stats(self) -> dict:
        st = md_stats()
        self._ck(lib.md_get_stats(self._h, ctypes.byref(st)))
        return st.as_dict()


def from_workload(w, precision: int | None = None, list_kind: int = MD_LIST_FULL, kernel: int = MD_KERNEL_TPA,
                  x=None, stream: int | None = None, options: dict | None = None) -> System:
    """Convenience: a System configured from a ``workloads.Workload`` (marshalling only)."""
    s = System(w.box, w.natoms, w.types, w.mass, stream=stream)
    s.md_set_units(w.ftm2v, w.mvv2e)
    s.md_set_precision(w.precision if precision is None else precision)
    s.md_set_neighbor(list_kind, kernel)
    for name, value in (options or {}).items():
        s.md_set_option(name, value)
    s.md_set_pair(w.style, w.params, w.rc, w.skin)
    if w.style == MD_PAIR_EAM_TAB:
        s.md_set_eam_tables(w.tables["rho_r"], w.tables["phi_r"], w.tables["F_rho"])
    if w.style == MD_PAIR_BUCK_COUL:
        nt = len(w.mass)
        for a in range(nt):
            for b in range(a, nt):
                s.md_set_pair_coeff(a, b, w.pair_coef[a][b])
        s.md_set_type_charges(w.qtype)
    s.md_set_positions(np.ascontiguousarray(w.x if x is None else x))
    s.md_set_velocities(np.ascontiguousarray(w.v))
    return s
