"""Pins of the oracle's velocity-Verlet NVE loop and its rebuild rule.

Closed forms and invariants only: the harmonic period of a bound LJ pair, time
reversal, second-order energy error, momentum conservation, and the fact that
the displacement-triggered Verlet list is an exact acceleration.
"""
import math

import numpy as np
import pytest

import oracle
from paper_1009_4330_b200 import workloads as wl

LJ = (1.0, 1.0)


def _period(mass, ftm2v, dt=0.0005, nsteps=6000):
    """Two atoms near the LJ minimum: period of r(t) from upward zero crossings of r - r_min."""
    r0 = 2.0 ** (1.0 / 6.0)
    box = np.array([10.0, 10.0, 10.0])
    x = np.array([[5.0, 5.0, 5.0], [5.0 + r0 + 1e-3, 5.0, 5.0]])
    v = np.zeros((2, 3))
    m = np.array([mass, mass])
    rs = []
    state_x, state_v = x, v
    for _ in range(nsteps):
        out = oracle.run_nve(state_x, state_v, box, m, oracle.PAIR_LJ, LJ, 2.5, 0.3, dt, 1, ftm2v=ftm2v)
        state_x, state_v = out["x"], out["v"]
        rs.append(state_x[1, 0] - state_x[0, 0] - r0)
    rs = np.array(rs)
    t = (np.arange(nsteps) + 1) * dt
    up = np.where((rs[:-1] < 0) & (rs[1:] >= 0))[0]
    tc = t[up] + dt * (-rs[up]) / (rs[up + 1] - rs[up])
    return float(np.mean(np.diff(tc)))


def test_bound_pair_period_mass_and_ftm2v():
    # u''(r_min) = 4 eps (156 r^-14 - 42 r^-8) = 72 * 2^(-1/3) eps/sigma^2 ; reduced mass m/2
    k = 72.0 * 2.0 ** (-1.0 / 3.0)
    for mass, ftm2v in [(1.0, 1.0), (2.0, 1.0), (1.0, 4.0)]:
        T = 2.0 * math.pi / math.sqrt(k * ftm2v / (mass / 2.0))
        assert _period(mass, ftm2v) == pytest.approx(T, rel=2e-4)


def _liquid(n=6, steps_melt=0):
    w = wl.make(1, n_override=n)
    return w


def test_time_reversal():
    w = _liquid()
    m = np.ones(w.natoms)
    a = oracle.run_nve(w.x, w.v, w.box, m, oracle.PAIR_LJ, LJ, 2.5, 0.3, 0.005, 40)
    b = oracle.run_nve(a["x"], -a["v"], w.box, m, oracle.PAIR_LJ, LJ, 2.5, 0.3, 0.005, 40)
    d = b["x"] - w.x
    d -= w.box * np.round(d / w.box)
    assert np.abs(d).max() < 1e-9
    assert np.abs(b["v"] + w.v).max() < 1e-8


def test_energy_error_is_second_order_and_momentum_conserved():
    """Cold crystal (T* = 0.01): rc = 2.5 sits between the 4th (2.375) and 5th (2.656) fcc shells, so no
    pair crosses the plain cutoff and the energy error is the integrator's alone: it must scale as dt^2."""
    w = _liquid()
    m = np.ones(w.natoms)
    v = w.v * math.sqrt(0.01 / 1.44)
    fl = []
    for dt, n in [(0.008, 100), (0.004, 200), (0.002, 400)]:
        out = oracle.run_nve(w.x, v, w.box, m, oracle.PAIR_LJ, LJ, 2.5, 0.3, dt, n, trace=True)
        e = out["pe"] + out["ke"]
        fl.append(np.abs(e - e[0]).max())
        p = (out["v"] * m[:, None]).sum(axis=0)
        assert np.abs(p).max() < 1e-11
        assert out["ke"][0] == pytest.approx(0.5 * (3 * w.natoms - 3) * 0.01, rel=1e-12)
    assert fl[0] / fl[1] == pytest.approx(4.0, rel=0.15)
    assert fl[1] / fl[2] == pytest.approx(4.0, rel=0.15)
    assert fl[2] < 1e-3 * 0.01 * w.natoms


def test_rebuild_rule_is_an_exact_acceleration():
    """Rebuilding every step (skin -> 0) or never needing to (huge skin) gives the same trajectory
    up to summation order: the list with skin is valid until the trigger fires."""
    w = _liquid()
    m = np.ones(w.natoms)
    ref = oracle.run_nve(w.x, w.v, w.box, m, oracle.PAIR_LJ, LJ, 2.5, 1e-9, 0.005, 60)
    assert ref["nbuild"] == 61
    for skin in (0.3, 0.6):
        out = oracle.run_nve(w.x, w.v, w.box, m, oracle.PAIR_LJ, LJ, 2.5, skin, 0.005, 60)
        assert 1 < out["nbuild"] < 30
        d = out["x"] - ref["x"]
        d -= w.box * np.round(d / w.box)
        assert np.abs(d).max() < 1e-10
        assert np.abs(out["f"] - ref["f"]).max() < 1e-8 * np.abs(ref["f"]).max()


def test_final_forces_belong_to_final_positions():
    w = _liquid()
    m = np.ones(w.natoms)
    out = oracle.run_nve(w.x, w.v, w.box, m, oracle.PAIR_LJ, LJ, 2.5, 0.3, 0.005, 25)
    fb = oracle.forces_brute(out["x"], w.box, oracle.PAIR_LJ, LJ, 2.5)[0]
    assert np.abs(out["f"] - fb).max() < 1e-11 * np.abs(fb).max()


def test_eam_metal_units_energy_conservation():
    """Cu crystal at 30 K in metal units (perfect lattice + thermal velocities: no pair reaches the plain
    cutoff, whose 4th shell is only 0.16 A outside, reading s12).  Total energy in eV is conserved only if
    ftm2v (force -> velocity) and mvv2e (velocity -> energy) are mutually consistent, and kinetic energy
    must flow into potential energy on the phonon time scale (~50 fs), which fixes their absolute size."""
    w = wl.make(4, n_override=5)
    x, _ = wl.fcc_lattice(5, wl.CU_A)
    m = np.full(w.natoms, w.mass[0])
    v = w.v * math.sqrt(30.0 / 300.0)
    out = oracle.run_nve(x, v, w.box, m, oracle.PAIR_EAM, w.params, w.rc, w.skin, w.dt, 100,
                         ftm2v=w.ftm2v, mvv2e=w.mvv2e, trace=True)
    e = (out["pe"] + out["ke"]) / w.natoms
    ke0 = out["ke"][0] / w.natoms
    assert ke0 == pytest.approx(1.5 * wl.KB_METAL * 30.0 * (w.natoms - 1) / w.natoms, rel=1e-12)
    assert 0.05 * ke0 < out["ke"].min() / w.natoms < 0.75 * ke0
    assert 20 <= int(np.argmin(out["ke"])) <= 99
    assert np.abs(e - e[0]).max() < 2e-4 * ke0
