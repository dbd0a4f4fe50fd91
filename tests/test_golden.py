"""Pins of the oracle against the text fixtures under tests/golden/ (each file cites its source).

paper_cost_model.txt holds the only numbers of this path the paper prints (App. C):
the ratio of atoms a 14-cell cell-list kernel reads to atoms inside the neighbor sphere.  The oracle's
brute-force pair enumeration on a seeded uniform gas must reproduce that ratio, which pins its distance
test (a wrong exponent, a missing component or r instead of r^2 changes the count by far more than 1 %).
"""
import math
import os

import numpy as np
import pytest

import oracle
from paper_1009_4330_b200 import workloads as wl

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _rows(name):
    out = []
    with open(os.path.join(GOLD, name)) as fh:
        for line in fh:
            line = line.split("#")[0].split()
            if line:
                out.append(line)
    return out


def test_paper_cost_model_ratio_from_oracle_counts():
    g = {r[0]: (float(r[1]), float(r[2])) for r in _rows("paper_cost_model.txt")}
    # the arithmetic the paper prints
    assert 14 * 3 / (4 * math.pi) == pytest.approx(g["ncell_over_nneigh"][0], abs=g["ncell_over_nneigh"][1])
    assert 42 / (4 * math.pi) == pytest.approx(g["alpha_limit_C3"][0], abs=g["alpha_limit_C3"][1])
    assert 1 - 4 * math.pi / 42 == pytest.approx(g["gamma_limit_C4"][0], abs=g["gamma_limit_C4"][1])
    assert (3 ** 3 - 1) // 2 + 1 == int(g["cells_read"][0])
    # the same ratio from the oracle: uniform gas, c = 1.5, box 9 = 6 c
    N, L, c = 6000, 9.0, 1.5
    ids = np.arange(N, dtype=np.uint64)
    x = np.stack([wl.uniform01(777, ids, k) for k in range(3)], axis=1) * L
    box = np.array([L, L, L])
    pi, _ = oracle.pairs_brute(x, box, c)
    n_neigh = 2.0 * len(pi) / N                       # atoms inside the sphere of radius c, per atom
    n_cell = 14 * c ** 3 * N / L ** 3                 # atoms in 14 cells of edge c at the same density
    assert n_neigh == pytest.approx(4.0 / 3.0 * math.pi * c ** 3 * N / L ** 3, rel=0.01)
    assert n_cell / n_neigh == pytest.approx(g["alpha_limit_C3"][0], rel=0.01)
    cnt, _ = oracle.neighbors_sample(x, box, c, np.arange(0, N, 7), stride=256)
    assert cnt.mean() == pytest.approx(n_neigh, rel=0.03)


def test_lj_pair_values_file():
    for r, u, F in _rows("lj_pair_values.txt"):
        r, u, F = float(r), float(u), float(F)
        L = max(10.0, 4.0 * r)
        box = np.array([L, L, L])
        x = np.array([[1.0 + r, 2.0, 3.0], [1.0, 2.0, 3.0]])
        f, E, W, npairs, _ = oracle.forces_brute(x, box, oracle.PAIR_LJ, (1.0, 1.0), r + 0.5)
        assert npairs == 1
        assert E == pytest.approx(u, rel=1e-12, abs=1e-14)
        assert f[0, 0] == pytest.approx(F, rel=1e-12) and f[1, 0] == pytest.approx(-F, rel=1e-12)
        fs, es = oracle.forces_sample(x, box, oracle.PAIR_LJ, (1.0, 1.0), r + 0.5, np.array([0, 1]))
        assert fs[0, 0] == pytest.approx(F, rel=1e-12) and es.sum() == pytest.approx(u, rel=1e-12, abs=1e-14)


def test_fcc_lattice_sums_file():
    g = {r[0]: float(r[1]) for r in _rows("fcc_lattice_sums.txt")}
    w = wl.make(1, n_override=6)
    N = w.natoms
    _, E, W, npairs, _ = oracle.forces(w.x, w.box, oracle.PAIR_LJ, (1.0, 1.0), 2.5, skin=0.3)   # list route
    assert 2 * npairs == g["lj_rc2.5_neighbors"] * N
    assert E / N == pytest.approx(g["lj_rc2.5_pe_per_atom"], abs=1e-10)
    assert W[:3].sum() / N == pytest.approx(g["lj_rc2.5_virial_per_atom"], abs=1e-10)
    start, _ = oracle.NeighborList(w.x, w.box, 2.8).csr()
    assert np.all(np.diff(start) == g["lj_rc2.5_list_neighbors"])
    x, box = wl.fcc_lattice(5, wl.CU_A)
    _, E, _, npairs, rho = oracle.forces(x, box, oracle.PAIR_EAM, wl.EAM_PARAMS, 4.95, skin=1.0)
    assert 2 * npairs == g["eam_neighbors"] * 500
    assert np.allclose(rho, g["eam_rho"], atol=1e-9)
    assert E / 500 == pytest.approx(g["eam_e_per_atom"], abs=1e-9)
