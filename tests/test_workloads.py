"""The seeded input generator: shapes, determinism and the statistics the configs promise."""
import numpy as np
import pytest

from paper_1009_4330_b200 import workloads as wl


def test_counter_based_rng_is_order_independent_and_uniform():
    ids = np.arange(200000, dtype=np.uint64)
    u = wl.uniform01(7, ids, 3)
    assert np.array_equal(u[::-1], wl.uniform01(7, ids[::-1], 3))
    assert 0.0 <= u.min() and u.max() < 1.0
    assert abs(u.mean() - 0.5) < 3e-3 and abs(u.var() - 1.0 / 12.0) < 2e-3
    assert not np.array_equal(u, wl.uniform01(8, ids, 3))
    assert not np.array_equal(u, wl.uniform01(7, ids, 4))
    g = wl.gaussian(7, ids, 0)
    assert abs(g.mean()) < 0.01 and abs(g.std() - 1.0) < 0.01
    assert abs(np.corrcoef(g, wl.gaussian(7, ids, 1))[0, 1]) < 0.01


@pytest.mark.parametrize("cfg,n,natoms", [(1, 10, 4000), (2, 20, 32000), (4, 6, 864), (5, 8, 2048)])
def test_config_shapes_and_state_point(cfg, n, natoms):
    w = wl.make(cfg, n_override=n)
    assert w.natoms == natoms and w.x.shape == (natoms, 3) and w.v.shape == (natoms, 3)
    assert np.all(w.x >= 0.0) and np.all(w.x < w.box)
    m = w.mass[0]
    assert np.abs((m * w.v).sum(axis=0)).max() < 1e-9 * natoms
    ke = 0.5 * w.mvv2e * m * (w.v ** 2).sum()
    assert ke == pytest.approx(0.5 * (3 * natoms - 3) * w.kT, rel=1e-12)
    if w.style == wl.PAIR_LJ:
        assert natoms / np.prod(w.box) == pytest.approx(0.8442, rel=1e-12)
    else:
        assert natoms / np.prod(w.box) == pytest.approx(0.0847, abs=1e-4)
    again = wl.make(cfg, n_override=n)
    assert np.array_equal(again.x, w.x) and np.array_equal(again.v, w.v)


def test_cfg5_is_a_permutation_of_the_lattice():
    w = wl.make(5, n_override=6)
    x, _ = wl.fcc_lattice(6, wl.LJ_A)
    p = wl.permutation(w.seed, len(x))
    assert sorted(p.tolist()) == list(range(len(x)))
    assert np.array_equal(w.x, x[p])
    assert np.abs(np.diff(p)).mean() > len(x) / 6          # really shuffled, not a rotation


def test_replicas_differ():
    a, b = wl.make(2, n_override=6), wl.make(2, n_override=6, seed_offset=1)
    assert np.array_equal(a.x, b.x) and not np.array_equal(a.v, b.v)
