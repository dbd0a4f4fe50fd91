"""Pins of the oracle's NVT integrator ("NVE, NVT, and NPT integrators"; reading s25: one
Nose-Hoover thermostat, symmetric splitting TH(dt/2) kick drift force kick TH(dt/2)) against things other than itself:

  * tau -> infinity switches the thermostat off: the trajectory is the NVE one (pinned in test_oracle_nve.py);
  * free particles (no forces): KE and xi obey the two-variable ODE dKE/dt = -2 xi KE, dxi/dt = (2 KE - g kT)/Q, which
    scipy integrates to 1e-10 independently;
  * time reversal: n steps, negate v and xi, n steps -> the initial state;
  * the conserved quantity H = KE + PE + Q xi^2/2 + g kT eta on a soft-sphere fluid whose pair energy vanishes at the cutoff: bounded
    fluctuation that falls 4x when dt is halved (second order), no drift;
  * the temperature settles at the target.
"""
import numpy as np
import pytest
from scipy.integrate import solve_ivp

import oracle
from paper_1009_4330_b200 import workloads as wl


def _cu(n=5):
    w = wl.make(4, n_override=n)        # EAM Cu crystal, metal units, 300 K: rc = 4.95 A lies between the 3rd and 4th shell
    return w, np.full(w.natoms, w.mass[0])


def test_infinite_damping_time_is_nve():
    w = wl.make(1, n_override=6)
    m = np.ones(w.natoms)
    a = oracle.run_nve(w.x, w.v, w.box, m, w.style, w.params, w.rc, w.skin, w.dt, 40)
    b = oracle.run_nvt(w.x, w.v, w.box, m, w.style, w.params, w.rc, w.skin, w.dt, 40, kT=0.7, tau=1e30)
    assert np.abs(a["x"] - b["x"]).max() < 1e-13 and np.abs(a["v"] - b["v"]).max() < 1e-13 and a["nbuild"] == b["nbuild"]
    assert abs(b["thermo"][0]) < 1e-40


def test_free_particles_follow_the_thermostat_ode():
    w = wl.make(1, n_override=6)
    m = np.ones(w.natoms)
    kT, tau, dt, n = 0.9, 0.4, 0.002, 1500
    g = 3 * w.natoms - 3
    Q = g * kT * tau * tau
    r = oracle.run_nvt(w.x, w.v, w.box, m, w.style, (0.0, 1.0), w.rc, w.skin, dt, n, kT=kT, tau=tau)     # eps = 0: no forces
    ke0 = 0.5 * (w.v ** 2).sum()
    sol = solve_ivp(lambda t, y: [-2.0 * y[1] * y[0], (2.0 * y[0] - g * kT) / Q], (0.0, n * dt), [ke0, 0.0],
                    rtol=1e-11, atol=1e-11, t_eval=[n * dt / 3, 2 * n * dt / 3, n * dt], method="DOP853")
    for k, step in enumerate([n // 3, 2 * n // 3, n]):
        assert r["ke"][step] == pytest.approx(sol.y[0][k], rel=2e-5)           # splitting error O(dt^2)
    assert r["thermo"][0] == pytest.approx(sol.y[1][-1], rel=2e-5, abs=1e-7)
    # second order: halving dt quarters the error
    r2 = oracle.run_nvt(w.x, w.v, w.box, m, w.style, (0.0, 1.0), w.rc, w.skin, dt / 2, 2 * n, kT=kT, tau=tau)
    e1, e2 = abs(r["ke"][n] - sol.y[0][-1]), abs(r2["ke"][2 * n] - sol.y[0][-1])
    assert e1 / e2 == pytest.approx(4.0, rel=0.15)
    # the oscillation is a real one: the temperature crosses the target
    T = 2 * r["ke"] / g
    assert T.min() < kT < T.max()


def test_time_reversal():
    w, m = _cu()
    kw = dict(ftm2v=w.ftm2v, mvv2e=w.mvv2e)
    kT2 = 2.0 * w.kT
    a = oracle.run_nvt(w.x, w.v, w.box, m, w.style, w.params, w.rc, w.skin, w.dt, 40, kT=kT2, tau=0.02, **kw)
    b = oracle.run_nvt(a["x"], -a["v"], w.box, m, w.style, w.params, w.rc, w.skin, w.dt, 40, kT=kT2, tau=0.02,
                       thermo=(-a["thermo"][0], a["thermo"][1]), **kw)
    d = b["x"] - w.x
    d -= w.box * np.round(d / w.box)
    assert np.abs(d).max() < 1e-10 and np.abs(b["v"] + w.v).max() < 1e-9 * np.abs(w.v).max()
    assert abs(b["thermo"][0]) < 1e-9 * abs(a["thermo"][0])


def _soft_spheres():
    """A purely repulsive exponential fluid (the Buckingham style with C = 0, q = 0) whose pair energy at the cutoff is
    4e-6: pairs crossing the cutoff do not disturb the energy balance (LJ and EAM are truncated plainly: they do)."""
    w = wl.make(1, n_override=6)
    P = dict(k=0.0, types=np.zeros(w.natoms, np.int32), q=[0.0], coef=np.array([[[2000.0, 0.15, 0.0]]]))
    return w, np.ones(w.natoms), P, 3.0


def test_conserved_quantity_is_second_order_and_does_not_drift():
    w, m, P, rc = _soft_spheres()
    kT2, tau = 0.7, 0.2
    h = {}
    for dt, n in [(0.004, 500), (0.002, 1000)]:
        r = oracle.run_nvt(w.x, w.v, w.box, m, oracle.PAIR_BUCK_COUL, P, rc, w.skin, dt, n, kT=kT2, tau=tau)
        h[dt] = r["h"] - r["h"][0]
        assert abs(r["thermo"][0]) > 0 and r["ke"].min() < 0.7 * r["ke"][0]          # the thermostat is doing work (1.44 -> 0.7)
    amp1, amp2 = np.abs(h[0.004]).max(), np.abs(h[0.002]).max()
    ke_scale = 1.5 * w.natoms * kT2
    assert amp1 < 1e-3 * ke_scale                                   # bounded, tiny against the energy the thermostat moved
    assert amp1 / amp2 == pytest.approx(4.0, rel=0.4)               # second order
    assert abs(h[0.002][-250:].mean() - h[0.002][250:500].mean()) < amp2            # no drift


def test_temperature_settles_at_the_target():
    w, m = _cu(5)
    g = 3 * w.natoms - 3
    kT2 = 2.0 * w.kT                                # 600 K from a 300 K start
    r = oracle.run_nvt(w.x, w.v, w.box, m, w.style, w.params, w.rc, w.skin, 0.002, 3000, kT=kT2, tau=0.05,
                       ftm2v=w.ftm2v, mvv2e=w.mvv2e)
    T = 2 * r["ke"] / g
    assert T[0] == pytest.approx(w.kT, rel=1e-12)
    assert T[1500:].mean() == pytest.approx(kT2, rel=0.03)
