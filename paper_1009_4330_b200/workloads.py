"""Seeded synthetic inputs for the five BASELINE.json configs.

This module serves BOTH the CPU oracle (``oracle/``) and the CUDA path.  It
holds none of the method's arithmetic: no forces, no neighbor search, no
integration.  It only lays atoms on an fcc lattice, draws counter-based random
numbers and scales velocities to a temperature (input preparation the paper
leaves to the LAMMPS input script, App. A).

The workloads stand in for the LAMMPS bench input decks and the tabulated Cu
EAM file the paper's runs used (neither is in the container); BASELINE.json's
analytic Finnis-Sinclair-style potential replaces the table.

Random numbers: counter-based, u = hash(seed, atom_id, stream) with SplitMix64
mixing -> 53-bit uniform; Gaussians by Box-Muller.  Order independent.
"""
from __future__ import annotations

import dataclasses
import math

import numpy as np

# metal units
KB_METAL = 8.617343e-5          # eV / K
MVV2E_METAL = 1.0364269e-4      # amu (A/ps)^2 -> eV
FTM2V_METAL = 1.0 / 1.0364269e-4

PAIR_LJ = 1
PAIR_EAM = 2
PAIR_BUCK_COUL = 3
PAIR_EAM_TAB = 4
PREC_FP64 = 0
PREC_MIXED = 1

_M64 = np.uint64(0xFFFFFFFFFFFFFFFF)
_GOLD = np.uint64(0x9E3779B97F4A7C15)
_C1 = np.uint64(0xBF58476D1CE4E5B9)
_C2 = np.uint64(0x94D049BB133111EB)
_STREAM_MUL = np.uint64(0xD1B54A32D192ED03)


def _splitmix64(z: np.ndarray) -> np.ndarray:
    """One SplitMix64 output step on an array of uint64 counters."""
    with np.errstate(over="ignore"):
        z = (z + _GOLD) & _M64
        z = ((z ^ (z >> np.uint64(30))) * _C1) & _M64
        z = ((z ^ (z >> np.uint64(27))) * _C2) & _M64
        return z ^ (z >> np.uint64(31))


def hash_u64(seed: int, ids: np.ndarray, stream: int) -> np.ndarray:
    """64-bit hash of (seed, atom id, stream)."""
    ids = np.asarray(ids, dtype=np.uint64)
    with np.errstate(over="ignore"):
        s = _splitmix64(np.full(1, seed, dtype=np.uint64))[0]
        k = (ids * _GOLD + np.uint64(stream) * _STREAM_MUL) & _M64
        return _splitmix64(_splitmix64(k ^ s))


def uniform01(seed: int, ids: np.ndarray, stream: int) -> np.ndarray:
    """Uniform in [0, 1) with 53 random bits."""
    return (hash_u64(seed, ids, stream) >> np.uint64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)


def gaussian(seed: int, ids: np.ndarray, stream: int) -> np.ndarray:
    """Standard normal by Box-Muller on streams (2*stream+16, 2*stream+17)."""
    u1 = uniform01(seed, ids, 2 * stream + 16)
    u2 = uniform01(seed, ids, 2 * stream + 17)
    return np.sqrt(-2.0 * np.log1p(-u1)) * np.cos(2.0 * math.pi * u2)


def fcc_lattice(n: int, a: float) -> tuple[np.ndarray, np.ndarray]:
    """n x n x n fcc unit cells of edge a.  Atom index = ((iz*n+iy)*n+ix)*4+b.

    Returns (positions [4n^3, 3] float64, box [3])."""
    basis = np.array([[0.0, 0.0, 0.0], [0.5, 0.5, 0.0], [0.5, 0.0, 0.5], [0.0, 0.5, 0.5]])
    iz, iy, ix = np.meshgrid(np.arange(n), np.arange(n), np.arange(n), indexing="ij")
    cell = np.stack([ix.ravel(), iy.ravel(), iz.ravel()], axis=1).astype(np.float64)
    x = (cell[:, None, :] + basis[None, :, :]).reshape(-1, 3) * a
    return np.ascontiguousarray(x), np.array([n * a] * 3, dtype=np.float64)


def thermal_velocities(seed: int, ids: np.ndarray, mass: np.ndarray, kT: float, mvv2e: float) -> np.ndarray:
    """v ~ N(0, kT/m); subtract the centre-of-mass velocity; rescale so that
    sum 1/2 m v^2 * mvv2e = 1/2 (3N-3) kT exactly."""
    n = len(ids)
    v = np.stack([gaussian(seed, ids, c) for c in range(3)], axis=1)
    v *= np.sqrt(kT / (mass * mvv2e))[:, None]
    v -= (mass[:, None] * v).sum(axis=0) / mass.sum()
    ke = 0.5 * mvv2e * float((mass[:, None] * v * v).sum())
    v *= math.sqrt(0.5 * (3 * n - 3) * kT / ke)
    return np.ascontiguousarray(v)


def uniform_displacements(seed: int, ids: np.ndarray, amplitude: float) -> np.ndarray:
    """Each coordinate ~ U(-amplitude, +amplitude); streams 3..5."""
    return np.stack([(2.0 * uniform01(seed, ids, 3 + c) - 1.0) * amplitude for c in range(3)], axis=1)


def permutation(seed: int, n: int) -> np.ndarray:
    """Seeded permutation: sort atoms by their 64-bit key (stream 6), ties by id."""
    key = hash_u64(seed, np.arange(n, dtype=np.uint64), 6)
    return np.lexsort((np.arange(n), key))


@dataclasses.dataclass
class Workload:
    name: str
    cfg: int
    x: np.ndarray            # [N,3] float64, inside [0,L)
    v: np.ndarray            # [N,3] float64
    box: np.ndarray          # [3]
    types: np.ndarray        # [N] int32 (all zero: single species)
    mass: np.ndarray         # [ntypes]
    style: int
    params: tuple            # LJ: (eps, sigma); EAM: (A, p, B, q, r0)
    rc: float
    skin: float
    dt: float
    nsteps: int
    precision: int
    ftm2v: float
    mvv2e: float
    kT: float
    seed: int
    qtype: np.ndarray | None = None       # PAIR_BUCK_COUL: charge of every type
    pair_coef: np.ndarray | None = None   # PAIR_BUCK_COUL: [ntypes, ntypes, 3] = A, rho, C of every type pair (symmetric)
    tables: dict | None = None            # PAIR_EAM_TAB: dict(dr, drho, rho_r, phi_r, F_rho)

    @property
    def natoms(self) -> int:
        return int(self.x.shape[0])


LJ_RHO = 0.8442
LJ_A = (4.0 / LJ_RHO) ** (1.0 / 3.0)
CU_A = 3.615
EAM_PARAMS = (0.0855, 10.96, 1.2240, 2.278, 2.556)   # A[eV], p, B[eV], q, r0[A]  (BASELINE.json cfg 4)

# cfg -> (style, n_cells, rc, skin, dt, nsteps, precision, permuted)
_TABLE = {
    1: ("LJ 12-6 fluid 4,000 atoms fp64", PAIR_LJ, 10, 2.5, 0.3, 0.005, 100, PREC_FP64, False),
    2: ("LJ 12-6 fluid 32,000 atoms mixed", PAIR_LJ, 20, 2.5, 0.3, 0.005, 1000, PREC_MIXED, False),
    3: ("LJ 12-6 fluid 256,000 atoms rc=5.0 mixed", PAIR_LJ, 40, 5.0, 0.3, 0.005, 500, PREC_MIXED, False),
    4: ("EAM Cu 256,000 atoms mixed", PAIR_EAM, 40, 4.95, 1.0, 0.001, 500, PREC_MIXED, False),
    5: ("LJ 12-6 liquid 4,000,000 atoms permuted mixed", PAIR_LJ, 100, 2.5, 0.3, 0.005, 200, PREC_MIXED, True),
}


# cfg 6: a synthetic stand-in for the paper's "silicate (cutoff)" workload (App. A: buck/coul/cut,
# 0.09 atoms per A^3, two charged species), whose data file and parameters are not in the container.  Rock-salt sites of
# spacing 2.25 A (0.0878 per A^3), anions (type 0) and cations (type 1) alternating, seeded displacements of 0.1 A;
# Buckingham coefficients of the magnitude of the BKS silica potential.  rc = 8 A, not the paper's 15 A: a cell of edge
# rc + skin must hold fewer than 8191/27 atoms for the tile's 16-bit slot codes (known limits).
K_COULOMB_METAL = 14.399645             # eV A / e^2
SILICATE_A0 = 2.25
SILICATE_Q = (-1.2, 1.2)
SILICATE_MASS = (15.9994, 28.0855)
SILICATE_COEF = {(0, 0): (1388.77, 0.3623, 175.0), (0, 1): (18003.76, 0.2052, 133.54), (1, 1): (0.0, 1.0, 0.0)}


def make_silicate_like(n: int = 48, seed_offset: int = 0, rc: float = 8.0, skin: float = 1.0, nsteps: int = 100) -> Workload:
    seed = 43306 + 1000 * seed_offset
    iz, iy, ix = np.meshgrid(np.arange(n), np.arange(n), np.arange(n), indexing="ij")
    site = np.stack([ix.ravel(), iy.ravel(), iz.ravel()], axis=1)
    types = ((site.sum(axis=1)) % 2).astype(np.int32)
    box = np.array([n * SILICATE_A0] * 3, dtype=np.float64)
    N = site.shape[0]
    ids = np.arange(N, dtype=np.uint64)
    x = site.astype(np.float64) * SILICATE_A0 + uniform_displacements(seed, ids, 0.1)
    x -= np.floor(x / box) * box
    mass = np.array(SILICATE_MASS)
    kT = KB_METAL * 300.0
    v = thermal_velocities(seed, ids, mass[types], kT, MVV2E_METAL)
    coef = np.zeros((2, 2, 3))
    for (a, b), c in SILICATE_COEF.items():
        coef[a, b] = coef[b, a] = c
    return Workload(name="Buckingham + cutoff Coulomb, two species, %d atoms mixed" % N, cfg=6, x=np.ascontiguousarray(x), v=v, box=box,
                    types=types, mass=mass, style=PAIR_BUCK_COUL, params=(K_COULOMB_METAL,), rc=rc, skin=skin, dt=0.001, nsteps=nsteps,
                    precision=PREC_MIXED, ftm2v=FTM2V_METAL, mvv2e=MVV2E_METAL, kT=kT, seed=seed, qtype=np.array(SILICATE_Q), pair_coef=coef)


def make_eam_tabulated(n_cells: int = 40, n_table: int = 2001, rmax: float = 6.0, rhomax: float = 60.0, seed_offset: int = 0) -> Workload:
    """cfg 4 with its potential given as TABLES (App. A: the paper's EAM run read a tabulated
    Cu potential file, which is not in the container): the Finnis-Sinclair functions of BASELINE.json cfg 4 sampled on
    ``n_table`` points of [0, rmax] A and [0, rhomax].  An input table, like the lattice: the interpolation is the method's."""
    w = make(4, n_override=n_cells, seed_offset=seed_offset)
    A, p, B, q, r0 = EAM_PARAMS
    dr, drho = rmax / (n_table - 1), rhomax / (n_table - 1)
    r, rh = np.arange(n_table) * dr, np.arange(n_table) * drho
    tables = dict(dr=dr, drho=drho, rho_r=np.exp(-q * (r / r0 - 1.0)), phi_r=A * np.exp(-p * (r / r0 - 1.0)), F_rho=-B * np.sqrt(rh))
    return dataclasses.replace(w, name="EAM Cu tabulated (%d-point tables) %d atoms mixed" % (n_table, w.natoms), cfg=7, style=PAIR_EAM_TAB,
                               params=(dr, drho), tables=tables)


def oracle_params(w: Workload):
    """The pair parameters of ``w`` in the form the CPU oracle's wrapper takes them (packing only)."""
    if w.style == PAIR_BUCK_COUL:
        return dict(k=w.params[0], types=w.types, q=w.qtype, coef=w.pair_coef)
    if w.style == PAIR_EAM_TAB:
        return w.tables
    return w.params


def make(cfg: int, n_override: int | None = None, seed_offset: int = 0) -> Workload:
    """Build config ``cfg`` (1..5) of BASELINE.json (6: the synthetic two-species workload of SURVEY.md 8(f)-2).  ``n_override`` shrinks the
    lattice (unit cells per edge) for tests; ``seed_offset`` decorrelates replicas."""
    if cfg == 7:
        return make_eam_tabulated(40 if n_override is None else int(n_override), seed_offset=seed_offset)
    if cfg == 6:
        return make_silicate_like(48 if n_override is None else int(n_override), seed_offset)
    name, style, n, rc, skin, dt, nsteps, prec, permuted = _TABLE[cfg]
    if n_override is not None:
        n = int(n_override)
    seed = 43300 + cfg + 1000 * seed_offset
    if style == PAIR_LJ:
        x, box = fcc_lattice(n, LJ_A)
        mass = np.array([1.0])
        kT, ftm2v, mvv2e = 1.44, 1.0, 1.0
        params = (1.0, 1.0)
    else:
        x, box = fcc_lattice(n, CU_A)
        mass = np.array([63.55])
        kT, ftm2v, mvv2e = KB_METAL * 300.0, FTM2V_METAL, MVV2E_METAL
        params = EAM_PARAMS
    N = x.shape[0]
    ids = np.arange(N, dtype=np.uint64)
    if style == PAIR_EAM:
        x = x + uniform_displacements(seed, ids, 0.05)
        x -= np.floor(x / box) * box
    v = thermal_velocities(seed, ids, np.full(N, mass[0]), kT, mvv2e)
    if permuted:
        p = permutation(seed, N)
        x, v = np.ascontiguousarray(x[p]), np.ascontiguousarray(v[p])
    return Workload(name=name, cfg=cfg, x=x, v=v, box=box, types=np.zeros(N, dtype=np.int32), mass=mass,
                    style=style, params=params, rc=rc, skin=skin, dt=dt, nsteps=nsteps, precision=prec,
                    ftm2v=ftm2v, mvv2e=mvv2e, kT=kT, seed=seed)


def perturbed(w: Workload, amplitude: float, seed: int = 7) -> np.ndarray:
    """Positions of ``w`` with seeded uniform displacements, wrapped into the box.
    Force-parity snapshots need this: a perfect lattice has zero net force
    (SURVEY.md §7 hard part 7)."""
    ids = np.arange(w.natoms, dtype=np.uint64)
    x = w.x + uniform_displacements(seed, ids, amplitude)
    x -= np.floor(x / w.box) * w.box
    return np.ascontiguousarray(x)
