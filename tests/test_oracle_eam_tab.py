"""Pins of the oracle's tabulated EAM style ("then tabulated/spline EAM (what the paper's EAM run actually
used)"; App. A; reading s26: rho(r), phi(r), F(rho) on uniform grids, cubic Hermite interpolation with
centred-difference node slopes, forces from the derivative of the interpolant) against things other than itself:

  * tables sampled from the analytic Finnis-Sinclair functions converge to the analytic EAM oracle (itself pinned by
    lattice sums and closed forms) as h^4;
  * tables of CUBIC polynomials are reproduced exactly: the energy equals a direct evaluation of the polynomials over
    the brute-force pair list (an independent composition of E = sum F(rho_i) + sum phi);
  * forces and virial are the exact gradient of the interpolated energy (finite differences), Newton's third law;
  * the list route and the sampled scans equal the O(N^2) route.
"""
import numpy as np
import pytest

import oracle
from paper_1009_4330_b200 import workloads as wl


def fs_tables(w, n, rmax=6.0, rhomax=60.0):
    A, p, B, q, r0 = w.params
    dr, drho = rmax / (n - 1), rhomax / (n - 1)
    r, rh = np.arange(n) * dr, np.arange(n) * drho
    return dict(dr=dr, drho=drho, rho_r=np.exp(-q * (r / r0 - 1)), phi_r=A * np.exp(-p * (r / r0 - 1)), F_rho=-B * np.sqrt(rh))


def crystal(n=5, amp=0.15):
    w = wl.make(4, n_override=n)
    return w, wl.perturbed(w, amp)


def test_fine_tables_converge_to_the_analytic_potential_as_h4():
    w, x = crystal()
    fa, Ea, Wa, na, rhoa = oracle.forces_brute(x, w.box, oracle.PAIR_EAM, w.params, w.rc)
    err = {}
    for n in (301, 601, 1201):
        ft, Et, Wt, nt, rhot = oracle.forces_brute(x, w.box, oracle.PAIR_EAM_TAB, fs_tables(w, n), w.rc)
        assert nt == na
        err[n] = (abs(Et - Ea) / abs(Ea), np.abs(ft - fa).max() / np.abs(fa).max(), np.abs(rhot - rhoa).max() / rhoa.max())
    assert err[1201][0] < 1e-10 and err[1201][1] < 2e-7 and err[1201][2] < 1e-10
    # fourth order in the grid spacing for the values (energy, density), third for the derivative (forces)
    assert err[301][0] / err[601][0] == pytest.approx(16.0, rel=0.35)
    assert err[301][2] / err[601][2] == pytest.approx(16.0, rel=0.35)
    assert 6.0 < err[301][1] / err[601][1] < 20.0


def test_cubic_tables_are_reproduced_exactly():
    w, x = crystal()
    n = 121
    dr, drho = 6.0 / (n - 1), 60.0 / (n - 1)
    r, rh = np.arange(n) * dr, np.arange(n) * drho
    rho_poly = np.poly1d([-0.004, 0.09, -0.62, 2.1])      # positive and decreasing on [2, 5]
    phi_poly = np.poly1d([0.003, -0.02, -0.05, 0.4])
    F_poly = np.poly1d([1e-4, -0.004, -0.1, 0.2])
    P = dict(dr=dr, drho=drho, rho_r=rho_poly(r), phi_r=phi_poly(r), F_rho=F_poly(rh))
    f, E, W, npairs, rho = oracle.forces_brute(x, w.box, oracle.PAIR_EAM_TAB, P, w.rc)
    pi, pj, r2 = oracle.pairs_brute(x, w.box, w.rc, with_r2=True)
    d = np.sqrt(r2)
    assert d.min() > 4 * dr and d.max() < 6.0 - 4 * dr                     # away from the one-sided end stencils
    rho_ref = np.zeros(len(x))
    np.add.at(rho_ref, pi, rho_poly(d)); np.add.at(rho_ref, pj, rho_poly(d))
    assert rho_ref.min() > 4 * drho and rho_ref.max() < 60.0 - 4 * drho
    assert np.abs(rho - rho_ref).max() < 1e-12 * rho_ref.max()
    assert E == pytest.approx(F_poly(rho_ref).sum() + phi_poly(d).sum(), rel=1e-12)
    # the force on one atom, written out from the definition with the polynomials' own derivatives
    i = 17
    Fp = F_poly.deriv()(rho_ref)
    fi = np.zeros(3)
    for a, b, dist in zip(pi, pj, d):
        if a == i or b == i:
            j = b if a == i else a
            D = x[i] - x[j]
            D -= w.box * np.round(D / w.box)
            fi += -((Fp[i] + Fp[j]) * rho_poly.deriv()(dist) + phi_poly.deriv()(dist)) * D / dist
    assert np.abs(f[i] - fi).max() < 1e-11 * np.abs(f).max()


def test_forces_and_virial_are_the_gradient_of_the_interpolated_energy():
    w, x = crystal()
    P = fs_tables(w, 61)                    # a COARSE table: the interpolant differs from the analytic function, its gradient must not
    d_all = np.sqrt(oracle.pairs_brute(x, w.box, w.rc + 0.05, with_r2=True)[2])
    rc = next(c for c in w.rc - 0.003 * np.arange(30) if np.abs(d_all - c).min() > 2e-4)     # no pair crosses the cutoff below
    f, E, W = oracle.forces_brute(x, w.box, oracle.PAIR_EAM_TAB, P, rc)[:3]
    h = 1e-5
    rng = np.random.default_rng(5)
    for i in rng.choice(len(x), 5, replace=False):
        for a in range(3):
            xp, xm = x.copy(), x.copy()
            xp[i, a] += h; xm[i, a] -= h
            Ep = oracle.forces_brute(xp, w.box, oracle.PAIR_EAM_TAB, P, rc)[1]
            Em = oracle.forces_brute(xm, w.box, oracle.PAIR_EAM_TAB, P, rc)[1]
            assert f[i, a] == pytest.approx(-(Ep - Em) / (2 * h), rel=3e-6, abs=3e-7)   # the interpolant is C1: its curvature jumps at the nodes
    for a in range(3):
        sp = np.ones(3); sp[a] += h
        sm = np.ones(3); sm[a] -= h
        Ep = oracle.forces_brute(x * sp, w.box * sp, oracle.PAIR_EAM_TAB, P, rc)[1]
        Em = oracle.forces_brute(x * sm, w.box * sm, oracle.PAIR_EAM_TAB, P, rc)[1]
        assert W[a] == pytest.approx(-(Ep - Em) / (2 * h), rel=1e-6, abs=1e-6)
    assert np.abs(f.sum(0)).max() < 1e-10 * np.abs(f).max() * len(x)
    # and the coarse interpolant really is a different function from the analytic one
    fa = oracle.forces_brute(x, w.box, oracle.PAIR_EAM, w.params, rc)[0]
    assert np.abs(f - fa).max() > 1e-5 * np.abs(fa).max()


def test_list_route_and_sampled_scans_match_brute_force():
    w, x = crystal(6)
    P = fs_tables(w, 401)
    fb, Eb, Wb, nb, rb = oracle.forces_brute(x, w.box, oracle.PAIR_EAM_TAB, P, w.rc)
    fl, El, Wl, nl, rl = oracle.forces(x, w.box, oracle.PAIR_EAM_TAB, P, w.rc, skin=w.skin)
    assert nl == nb and El == pytest.approx(Eb, rel=1e-12) and np.abs(rl - rb).max() < 1e-12 * rb.max()
    assert np.abs(fl - fb).max() < 1e-11 * np.abs(fb).max() and np.allclose(Wl, Wb, rtol=1e-10, atol=1e-9)
    ids = np.array([0, 33, 500, len(x) - 1])
    fs, es = oracle.forces_sample(x, w.box, oracle.PAIR_EAM_TAB, P, w.rc, ids)
    assert np.abs(fs - fb[ids]).max() < 1e-11 * np.abs(fb).max()
