"""ctypes face of ``oracle/md_oracle.c`` -- TEST INFRASTRUCTURE, not the product.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s cpu_baseline /
``--impl reference`` legs may import this package.  It never imports the CUDA
path (``paper_1009_4330_b200``) and shares no code with it.

``build()`` compiles the C file with gcc (``-O2 -fopenmp``) into
``oracle/liboracle.so``; importing the package builds it when missing or stale.
Every function below cites the passage of PAPER.md / SURVEY.md it follows in
the C source.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "md_oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")

PAIR_LJ = 1
PAIR_EAM = 2
PAIR_EAM_TAB = 4     # params: dict(dr, drho, rho_r=float[nr], phi_r=float[nr], F_rho=float[nrho]): tables on uniform grids from 0
PAIR_BUCK_COUL = 3   # params: dict(k=Coulomb constant, types=int32[N], q=float[ntypes], coef=float[ntypes, ntypes, 3] = A, rho, C)


def build(force: bool = False) -> str:
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".tmp%d" % os.getpid()
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-fno-fast-math", "-ffp-contract=off", "-shared", "-fPIC",
                               "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


class _Pair(ctypes.Structure):
    _fields_ = [("style", ctypes.c_int), ("p", ctypes.c_double * 5), ("rc", ctypes.c_double),
                ("type", ctypes.POINTER(ctypes.c_int32)), ("ntypes", ctypes.c_int),
                ("coef", ctypes.POINTER(ctypes.c_double)), ("qtype", ctypes.POINTER(ctypes.c_double)),
                ("nr", ctypes.c_int), ("nrho", ctypes.c_int), ("dr", ctypes.c_double), ("drho", ctypes.c_double),
                ("tab_rho", ctypes.POINTER(ctypes.c_double)), ("tab_phi", ctypes.POINTER(ctypes.c_double)),
                ("tab_F", ctypes.POINTER(ctypes.c_double))]


def _pair(style: int, params, rc: float) -> _Pair:
    p = _Pair()
    p.style = int(style)
    p.rc = float(rc)
    if style == PAIR_BUCK_COUL:
        types = np.ascontiguousarray(params["types"], dtype=np.int32)
        q = np.ascontiguousarray(params["q"], dtype=np.float64)
        coef = np.ascontiguousarray(params["coef"], dtype=np.float64)
        nt = len(q)
        if coef.shape != (nt, nt, 3) or types.min() < 0 or types.max() >= nt:
            raise ValueError("buck/coul: coef must be [ntypes, ntypes, 3] and types must lie in 0..ntypes-1")
        if not np.array_equal(coef, coef.transpose(1, 0, 2)):
            raise ValueError("buck/coul: the coefficient table must be symmetric in the two types")
        p.p[0] = float(params["k"])
        p._keep = (types, q, coef)               # the struct only holds pointers
        p.type = types.ctypes.data_as(ctypes.POINTER(ctypes.c_int32))
        p.ntypes = nt
        p.coef = coef.ctypes.data_as(ctypes.POINTER(ctypes.c_double))
        p.qtype = q.ctypes.data_as(ctypes.POINTER(ctypes.c_double))
        return p
    if style == PAIR_EAM_TAB:
        rho_r = np.ascontiguousarray(params["rho_r"], dtype=np.float64)
        phi_r = np.ascontiguousarray(params["phi_r"], dtype=np.float64)
        F_rho = np.ascontiguousarray(params["F_rho"], dtype=np.float64)
        if len(rho_r) != len(phi_r) or len(rho_r) < 5 or len(F_rho) < 5:
            raise ValueError("tabulated EAM: rho_r and phi_r must have the same length >= 5, F_rho >= 5")
        p._keep = (rho_r, phi_r, F_rho)
        dp = ctypes.POINTER(ctypes.c_double)
        p.nr, p.nrho, p.dr, p.drho = len(rho_r), len(F_rho), float(params["dr"]), float(params["drho"])
        p.tab_rho, p.tab_phi, p.tab_F = rho_r.ctypes.data_as(dp), phi_r.ctypes.data_as(dp), F_rho.ctypes.data_as(dp)
        return p
    for k, val in enumerate(params):
        p.p[k] = float(val)
    return p


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = ctypes.CDLL(build())
        dp = ctypes.POINTER(ctypes.c_double)
        i32p = ctypes.POINTER(ctypes.c_int32)
        i64p = ctypes.POINTER(ctypes.c_int64)
        pp = ctypes.POINTER(_Pair)
        L.orc_max_threads.restype = ctypes.c_int
        L.orc_set_threads.argtypes = [ctypes.c_int]
        L.orc_pairs_brute.restype = ctypes.c_int64
        L.orc_pairs_brute.argtypes = [ctypes.c_int64, dp, dp, ctypes.c_double, i32p, i32p, dp, ctypes.c_int64]
        L.orc_forces_brute.argtypes = [ctypes.c_int64, dp, dp, pp, dp, dp, dp, i64p, dp]
        L.orc_forces_sample.argtypes = [ctypes.c_int64, dp, dp, pp, ctypes.c_int64, i64p, dp, dp]
        L.orc_neighbors_sample.argtypes = [ctypes.c_int64, dp, dp, ctypes.c_double, ctypes.c_int64, i64p, i32p, i32p,
                                           ctypes.c_int64]
        L.orc_list_build.restype = ctypes.c_void_p
        L.orc_list_build.argtypes = [ctypes.c_int64, dp, dp, ctypes.c_double]
        L.orc_list_free.argtypes = [ctypes.c_void_p]
        L.orc_list_total.restype = ctypes.c_int64
        L.orc_list_total.argtypes = [ctypes.c_void_p]
        L.orc_list_export.argtypes = [ctypes.c_void_p, i64p, i32p]
        L.orc_forces_list.argtypes = [ctypes.c_int64, dp, dp, pp, ctypes.c_void_p, dp, dp, dp, i64p, dp]
        L.orc_run_nve.restype = ctypes.c_int64
        L.orc_run_nve.argtypes = [ctypes.c_int64, dp, dp, dp, dp, dp, pp, ctypes.c_double, ctypes.c_double,
                                  ctypes.c_int64, ctypes.c_double, ctypes.c_double, dp, dp]
        _lib = L
    return _lib


def _d(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def _i32(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_int32))


def _i64(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_int64))


def _c(a, dtype=np.float64):
    return np.ascontiguousarray(a, dtype=dtype)


def max_threads() -> int:
    return int(lib().orc_max_threads())


def set_threads(n: int) -> None:
    lib().orc_set_threads(int(n))


def pairs_brute(x, box, rcut, with_r2=False):
    """All unordered pairs {i<j} with |mi(x_i-x_j)| < rcut, by the O(N^2) double loop."""
    x, box = _c(x), _c(box)
    N = x.shape[0]
    cap = max(1024, int(N * 64))
    while True:
        pi = np.empty(cap, np.int32)
        pj = np.empty(cap, np.int32)
        r2 = np.empty(cap, np.float64)
        n = lib().orc_pairs_brute(N, _d(x), _d(box), float(rcut), _i32(pi), _i32(pj), _d(r2), cap)
        if n <= cap:
            break
        cap = int(n)
    if with_r2:
        return pi[:n].copy(), pj[:n].copy(), r2[:n].copy()
    return pi[:n].copy(), pj[:n].copy()


def forces_brute(x, box, style, params, rc):
    """(f[N,3], E, W[6], npairs, rho[N] or None) by the O(N^2) double loop over i<j."""
    x, box = _c(x), _c(box)
    N = x.shape[0]
    f = np.zeros((N, 3))
    E = ctypes.c_double(0.0)
    W = np.zeros(6)
    npairs = ctypes.c_int64(0)
    rho = np.zeros(N) if style in (PAIR_EAM, PAIR_EAM_TAB) else None
    P = _pair(style, params, rc)
    lib().orc_forces_brute(N, _d(x), _d(box), ctypes.byref(P), _d(f), ctypes.byref(E), _d(W),
                           ctypes.byref(npairs), _d(rho) if rho is not None else None)
    return f, E.value, W, int(npairs.value), rho


def forces_sample(x, box, style, params, rc, ids):
    """Force on and energy share of the atoms ``ids``, each by a full scan over all atoms."""
    x, box = _c(x), _c(box)
    ids = _c(ids, np.int64)
    f = np.zeros((len(ids), 3))
    e = np.zeros(len(ids))
    P = _pair(style, params, rc)
    lib().orc_forces_sample(x.shape[0], _d(x), _d(box), ctypes.byref(P), len(ids), _i64(ids), _d(f), _d(e))
    return f, e


def neighbors_sample(x, box, rcut, ids, stride=1024):
    """Neighbor ids (ascending) of the atoms ``ids`` within rcut, each by a full scan."""
    x, box = _c(x), _c(box)
    ids = _c(ids, np.int64)
    cnt = np.zeros(len(ids), np.int32)
    nb = np.full((len(ids), stride), -1, np.int32)
    lib().orc_neighbors_sample(x.shape[0], _d(x), _d(box), float(rcut), len(ids), _i64(ids), _i32(cnt), _i32(nb),
                               stride)
    assert cnt.max(initial=0) <= stride
    return cnt, nb


class NeighborList:
    """Full Verlet list built through the oracle's own cell grid (CSR)."""

    def __init__(self, x, box, rl):
        self.x, self.box = _c(x), _c(box)
        self.N = self.x.shape[0]
        self._h = lib().orc_list_build(self.N, _d(self.x), _d(self.box), float(rl))
        if not self._h:
            raise ValueError("box smaller than 3 (rc+skin) in some dimension")

    def __del__(self):
        if getattr(self, "_h", None):
            lib().orc_list_free(self._h)
            self._h = None

    def csr(self):
        total = lib().orc_list_total(self._h)
        start = np.zeros(self.N + 1, np.int64)
        idx = np.zeros(max(total, 1), np.int32)
        lib().orc_list_export(self._h, _i64(start), _i32(idx))
        return start, idx[:total]

    def forces(self, x, style, params, rc):
        """(f, E, W, npairs, rho) through the list, at positions x (same atoms)."""
        x = _c(x)
        f = np.zeros((self.N, 3))
        E = ctypes.c_double(0.0)
        W = np.zeros(6)
        npairs = ctypes.c_int64(0)
        rho = np.zeros(self.N) if style in (PAIR_EAM, PAIR_EAM_TAB) else None
        P = _pair(style, params, rc)
        lib().orc_forces_list(self.N, _d(x), _d(self.box), ctypes.byref(P), self._h, _d(f), ctypes.byref(E), _d(W),
                              ctypes.byref(npairs), _d(rho) if rho is not None else None)
        return f, E.value, W, int(npairs.value), rho


def forces(x, box, style, params, rc, skin=0.0):
    """Forces via the O(N) route (cell grid + list of radius rc+skin)."""
    return NeighborList(x, box, rc + skin).forces(x, style, params, rc)


def run_nve(x, v, box, mass_per_atom, style, params, rc, skin, dt, nsteps, ftm2v=1.0, mvv2e=1.0, trace=False):
    """Velocity-Verlet NVE.  Returns dict(x, v, f, nbuild[, pe, ke])."""
    x, v, box, m = _c(x).copy(), _c(v).copy(), _c(box), _c(mass_per_atom)
    N = x.shape[0]
    f = np.zeros((N, 3))
    pe = np.zeros(nsteps + 1) if trace else None
    ke = np.zeros(nsteps + 1) if trace else None
    P = _pair(style, params, rc)
    nb = lib().orc_run_nve(N, _d(x), _d(v), _d(f), _d(box), _d(m), ctypes.byref(P), float(skin), float(dt),
                           int(nsteps), float(ftm2v), float(mvv2e), _d(pe) if trace else None,
                           _d(ke) if trace else None)
    if nb < 0:
        raise ValueError("box smaller than 3 (rc+skin) in some dimension")
    out = dict(x=x, v=v, f=f, nbuild=int(nb))
    if trace:
        out.update(pe=pe, ke=ke)
    return out


def run_nvt(x, v, box, mass_per_atom, style, params, rc, skin, dt, nsteps, kT, tau, ftm2v=1.0, mvv2e=1.0, thermo=(0.0, 0.0)):
    """Velocity Verlet with one Nose-Hoover thermostat (md_oracle.c header; reading s25).
    Returns dict(x, v, f, nbuild, thermo=(xi, eta), h[nsteps+1] conserved quantity, ke[nsteps+1])."""
    x, v, box, m = _c(x).copy(), _c(v).copy(), _c(box), _c(mass_per_atom)
    N = x.shape[0]
    f = np.zeros((N, 3))
    h = np.zeros(nsteps + 1)
    ke = np.zeros(nsteps + 1)
    th = np.array(thermo, dtype=np.float64)
    P = _pair(style, params, rc)
    L = lib()
    L.orc_run_nvt.restype = ctypes.c_int64
    dp = ctypes.POINTER(ctypes.c_double)
    L.orc_run_nvt.argtypes = [ctypes.c_int64, dp, dp, dp, dp, dp, ctypes.POINTER(_Pair), ctypes.c_double, ctypes.c_double,
                              ctypes.c_int64, ctypes.c_double, ctypes.c_double, ctypes.c_double, ctypes.c_double, dp, dp, dp]
    nb = L.orc_run_nvt(N, _d(x), _d(v), _d(f), _d(box), _d(m), ctypes.byref(P), float(skin), float(dt), int(nsteps),
                       float(ftm2v), float(mvv2e), float(kT), float(tau), _d(th), _d(h), _d(ke))
    if nb < 0:
        raise ValueError("box smaller than 3 (rc+skin) in some dimension")
    return dict(x=x, v=v, f=f, nbuild=int(nb), thermo=(float(th[0]), float(th[1])), h=h, ke=ke)
