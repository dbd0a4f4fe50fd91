"""Pins of the CPU oracle against things other than itself.

Nothing here touches the CUDA path.  The paper prints no force or energy of a
worked example, so the pins are closed forms, lattice sums done by direct
lattice-vector enumeration (a different algorithm from the oracle's periodic
min-image loops), finite differences, conservation laws and brute force.
"""
import math

import numpy as np
import pytest

import oracle
from paper_1009_4330_b200 import workloads as wl

LJ = (1.0, 1.0)
BOX10 = np.array([10.0, 10.0, 10.0])


def two_atoms(r, axis=0, box=BOX10, origin=(3.0, 4.0, 5.0)):
    x = np.array([origin, origin], dtype=np.float64)
    x[0, axis] += r
    return x


# ---- LJ pair function: analytic values (App. A, lj/cut) -----------------------------

@pytest.mark.parametrize("axis", [0, 1, 2])
def test_lj_two_atoms_analytic(axis):
    rmin = 2.0 ** (1.0 / 6.0)
    # u(sigma) = 0, F(sigma) = 24 eps / sigma (repulsive: pushes atom 0 along +axis)
    f, E, W, npairs, _ = oracle.forces_brute(two_atoms(1.0, axis), BOX10, oracle.PAIR_LJ, LJ, 3.0)
    assert npairs == 1
    assert abs(E) < 1e-14
    assert f[0, axis] == pytest.approx(24.0, rel=1e-14)
    assert f[1, axis] == pytest.approx(-24.0, rel=1e-14)
    assert np.abs(np.delete(f, axis, axis=1)).max() == 0.0
    # virial of one pair: W_aa = D_a * f_a = r * F
    assert W[axis] == pytest.approx(24.0, rel=1e-14)
    assert np.abs(np.delete(W, axis)).max() == 0.0
    # u(2^(1/6) sigma) = -eps, F = 0
    f, E, _, _, _ = oracle.forces_brute(two_atoms(rmin, axis), BOX10, oracle.PAIR_LJ, LJ, 3.0)
    assert E == pytest.approx(-1.0, rel=1e-14)
    assert np.abs(f).max() < 1e-13
    # u(2.5) = -0.016316891136 and F(2.5) = -0.0389994774528 (exact decimals of 4(r^-12 - r^-6))
    f, E, _, _, _ = oracle.forces_brute(two_atoms(2.5, axis), BOX10, oracle.PAIR_LJ, LJ, 3.0)
    assert E == pytest.approx(-0.016316891136, rel=1e-12)
    assert f[0, axis] == pytest.approx(-0.0389994774528, rel=1e-12)   # attractive: pulls atom 0 back
    # u(5.0) = -0.000255983616; L/2 = 10 > 5
    f, E, _, _, _ = oracle.forces_brute(two_atoms(5.0, axis, box=BOX10 * 2), BOX10 * 2, oracle.PAIR_LJ, LJ, 6.0)
    assert E == pytest.approx(-0.000255983616, rel=1e-12)


def test_lj_eps_sigma_scaling():
    # u_min = -eps at r = 2^(1/6) sigma for any eps, sigma
    eps, sigma = 2.0, 1.5
    x = two_atoms(sigma * 2.0 ** (1.0 / 6.0))
    f, E, _, _, _ = oracle.forces_brute(x, BOX10, oracle.PAIR_LJ, (eps, sigma), 4.0)
    assert E == pytest.approx(-eps, rel=1e-14)
    assert np.abs(f).max() < 1e-12
    f, E, _, _, _ = oracle.forces_brute(two_atoms(sigma), BOX10, oracle.PAIR_LJ, (eps, sigma), 4.0)
    assert f[0, 0] == pytest.approx(24.0 * eps / sigma, rel=1e-14)


def test_lj_cutoff_is_strict_and_plain():
    # plain truncation: nothing at or beyond rc (reading s3: r^2 < rc^2), unshifted inside
    for r, n in [(2.6, 0), (2.5, 0), (2.4999999, 1)]:
        f, E, _, npairs, _ = oracle.forces_brute(two_atoms(r), BOX10, oracle.PAIR_LJ, LJ, 2.5)
        assert npairs == n
        if n == 0:
            assert E == 0.0 and np.abs(f).max() == 0.0


def test_minimum_image_across_boundary():
    # atoms at 0.4 and L-0.6 are 1.0 apart through the periodic face; atom 0 is pushed in +x
    x = np.array([[0.4, 5.0, 5.0], [9.4, 5.0, 5.0]])
    f, E, _, npairs, _ = oracle.forces_brute(x, BOX10, oracle.PAIR_LJ, LJ, 2.5)
    assert npairs == 1 and abs(E) < 1e-13
    assert f[0, 0] == pytest.approx(24.0, rel=1e-12) and f[1, 0] == pytest.approx(-24.0, rel=1e-12)
    pi, pj = oracle.pairs_brute(x, BOX10, 2.8)
    assert list(zip(pi, pj)) == [(0, 1)]


# ---- perfect fcc: lattice sums by direct enumeration of lattice vectors ---------------------------

def fcc_shell_vectors(a, rcut):
    m = int(math.ceil(2.0 * rcut / a)) + 1
    out = []
    for i in range(-m, m + 1):
        for j in range(-m, m + 1):
            for k in range(-m, m + 1):
                if (i + j + k) % 2 == 0 and (i, j, k) != (0, 0, 0):
                    r2 = 0.25 * a * a * (i * i + j * j + k * k)
                    if r2 < rcut * rcut:
                        out.append(r2)
    return np.array(out)


@pytest.mark.parametrize("rc,nn,pe_survey,vir_survey", [
    (2.5, 54, -6.773368053253, -22.158199254035),
    (5.0, 428, -7.161692782477, -24.484683458322),
])
def test_lj_fcc_lattice_sums(rc, nn, pe_survey, vir_survey):
    """PE/atom, virial/atom and neighbor count of the rho*=0.8442 fcc crystal."""
    r2 = fcc_shell_vectors(wl.LJ_A, rc)
    assert len(r2) == nn
    s6 = 1.0 / r2 ** 3
    pe = float(np.sum(0.5 * 4.0 * (s6 * s6 - s6)))
    vir = float(np.sum(0.5 * 24.0 * (2.0 * s6 * s6 - s6)))        # 1/2 sum r . f
    assert pe == pytest.approx(pe_survey, abs=2e-11)
    assert vir == pytest.approx(vir_survey, abs=2e-11)
    w = wl.make(1, n_override=6)                                   # 864 atoms, L/2 = 5.039 > 5.0
    f, E, W, npairs, _ = oracle.forces_brute(w.x, w.box, oracle.PAIR_LJ, LJ, rc)
    N = w.natoms
    assert 2 * npairs == nn * N
    assert E / N == pytest.approx(pe, rel=1e-12)
    assert W[:3].sum() / N == pytest.approx(vir, rel=1e-12)
    assert W[0] == pytest.approx(W[1], rel=1e-12) and W[1] == pytest.approx(W[2], rel=1e-12)
    assert np.abs(W[3:]).max() < 1e-9 * abs(W[0])
    assert np.abs(f).max() < 1e-11                                 # every lattice site is a centre of symmetry
    # list radius: 78 entries at r_l = 2.8, 530 at 5.3 need L/2 > r_l: only the 2.8 case fits this box
    if rc == 2.5:
        pi, _ = oracle.pairs_brute(w.x, w.box, 2.8)
        assert 2 * len(pi) == 78 * N
    assert len(fcc_shell_vectors(wl.LJ_A, rc + 0.3)) == (78 if rc == 2.5 else 530)


def test_eam_fcc_lattice_sums():
    """Cu fcc a=3.615: 42 neighbors, rho, F(rho), 1/2 sum phi, E/atom, virial."""
    A, p, B, q, r0 = wl.EAM_PARAMS
    r = np.sqrt(fcc_shell_vectors(wl.CU_A, 4.95))
    assert len(r) == 42
    rho = float(np.sum(np.exp(-q * (r / r0 - 1.0))))
    half_phi = float(0.5 * np.sum(A * np.exp(-p * (r / r0 - 1.0))))
    assert rho == pytest.approx(18.8601872740, abs=1e-9)
    assert -B * math.sqrt(rho) == pytest.approx(-5.3156260148, abs=1e-9)
    assert half_phi == pytest.approx(0.5156509433, abs=1e-9)
    dF = -B / (2.0 * math.sqrt(rho))
    assert dF == pytest.approx(-0.1409218779, abs=1e-9)
    # dE/dln(r) per atom = sum_j r [F' rho' + 1/2 phi']  = +1.76240078 eV
    dEdlnr = float(np.sum(r * (dF * (-q / r0) * np.exp(-q * (r / r0 - 1.0))
                               + 0.5 * (-p / r0) * A * np.exp(-p * (r / r0 - 1.0)))))
    assert dEdlnr == pytest.approx(1.76240078, abs=1e-7)
    x, box = wl.fcc_lattice(5, wl.CU_A)                            # 500 atoms, L = 18.075
    f, E, W, npairs, rho_o = oracle.forces_brute(x, box, oracle.PAIR_EAM, wl.EAM_PARAMS, 4.95)
    assert 2 * npairs == 42 * 500
    assert np.allclose(rho_o, rho, rtol=1e-13)
    assert E / 500 == pytest.approx(-B * math.sqrt(rho) + half_phi, rel=5e-12)   # box coordinates carry ulp(18 A) rounding
    assert E / 500 == pytest.approx(-4.7999750715, abs=1e-9)
    assert W[:3].sum() / 500 == pytest.approx(-dEdlnr, rel=1e-12)
    assert np.abs(f).max() < 1e-12


def test_eam_isolated_atom_has_zero_embedding():
    # reading s13: an atom with no neighbor inside rc has rho = 0, F(0) = 0, F'(0) := 0 (no NaN)
    x = np.array([[1.0, 1.0, 1.0], [3.0, 1.0, 1.0], [10.0, 10.0, 10.0]])
    box = np.array([20.0, 20.0, 20.0])
    f, E, _, npairs, rho = oracle.forces_brute(x, box, oracle.PAIR_EAM, wl.EAM_PARAMS, 4.95)
    assert npairs == 1 and rho[2] == 0.0
    assert np.all(np.isfinite(f)) and np.all(f[2] == 0.0)
    A, p, B, q, r0 = wl.EAM_PARAMS
    g = math.exp(-q * (2.0 / r0 - 1.0))
    assert E == pytest.approx(2 * (-B * math.sqrt(g)) + A * math.exp(-p * (2.0 / r0 - 1.0)), rel=1e-13)


# ---- forces are minus the energy gradient; virial is minus the volume derivative -------------------

def _small_system(style, clear=0.0):
    """Perturbed small periodic system; the seed is advanced until no pair lies within ``clear`` of rc."""
    for seed in range(11, 40):
        if style == oracle.PAIR_LJ:
            w = wl.make(1, n_override=6)
            x, params, rc = wl.perturbed(w, 0.12, seed=seed), LJ, 2.5
        else:
            w = wl.make(4, n_override=5)
            x, params, rc = wl.perturbed(w, 0.25, seed=seed), wl.EAM_PARAMS, 4.95
        if clear > 0.0:
            _, _, r2 = oracle.pairs_brute(x, w.box, rc + 0.01, with_r2=True)
            if np.any(np.abs(np.sqrt(r2) - rc) < clear):
                continue
        return x, w.box, params, rc
    raise AssertionError("no seed keeps the cutoff shell clear")


def _energy(x, box, style, params, rc):
    return oracle.forces_brute(x, box, style, params, rc)[1]


@pytest.mark.parametrize("style", [oracle.PAIR_LJ, oracle.PAIR_EAM])
def test_forces_are_minus_energy_gradient(style):
    x, box, params, rc = _small_system(style)
    f, E, W, _, _ = oracle.forces_brute(x, box, style, params, rc)
    h = 1e-5
    # atoms with no pair within 4h of the cutoff (a crossing would put a jump into the difference quotient)
    pi, pj, r2 = oracle.pairs_brute(x, box, rc + 0.01, with_r2=True)
    near = np.abs(np.sqrt(r2) - rc) < 4 * h
    bad = set(pi[near]) | set(pj[near])
    atoms = [i for i in range(0, x.shape[0], 37) if i not in bad][:12]
    assert len(atoms) >= 8
    fscale = np.sqrt((f * f).sum(axis=1).mean())
    for i in atoms:
        for a in range(3):
            xp, xm = x.copy(), x.copy()
            xp[i, a] += h
            xm[i, a] -= h
            fd = -(_energy(xp, box, style, params, rc) - _energy(xm, box, style, params, rc)) / (2 * h)
            assert abs(fd - f[i, a]) < 2e-7 * fscale, (i, a, fd, f[i, a])


@pytest.mark.parametrize("style", [oracle.PAIR_LJ, oracle.PAIR_EAM])
def test_virial_is_minus_volume_derivative(style):
    h = 1e-6
    x, box, params, rc = _small_system(style, clear=4 * h * 5.0)
    _, _, W, _, _ = oracle.forces_brute(x, box, style, params, rc)
    dE = (_energy(x * (1 + h), box * (1 + h), style, params, rc)
          - _energy(x * (1 - h), box * (1 - h), style, params, rc)) / (2 * h)
    assert W[:3].sum() == pytest.approx(-dE, rel=2e-7)
    # off-diagonal and anisotropic parts: shear / uniaxial strain derivative, W_ab = -dE/d(eps_ab)
    for comp, (a, b) in zip(range(6), [(0, 0), (1, 1), (2, 2), (0, 1), (0, 2), (1, 2)]):
        if a == b:
            sp, sm = np.ones(3), np.ones(3)
            sp[a] += h
            sm[a] -= h
            dEab = (_energy(x * sp, box * sp, style, params, rc) - _energy(x * sm, box * sm, style, params, rc)) / (2 * h)
            assert W[comp] == pytest.approx(-dEab, rel=5e-7)


def test_newton_third_law_list_route():
    # the full-list route writes every f[i] on its own; the sum must still vanish
    for style in (oracle.PAIR_LJ, oracle.PAIR_EAM):
        x, box, params, rc = _small_system(style)
        f = oracle.forces(x, box, style, params, rc, skin=0.3)[0]
        assert np.abs(f.sum(axis=0)).max() < 1e-10 * np.abs(f).sum()


# ---- the O(N) list route equals the O(N^2) definition ----------------------------------------------

@pytest.mark.parametrize("style", [oracle.PAIR_LJ, oracle.PAIR_EAM])
def test_list_route_matches_brute_force(style):
    x, box, params, rc = _small_system(style)
    skin = 0.3 if style == oracle.PAIR_LJ else 1.0
    fb, Eb, Wb, nb, rhob = oracle.forces_brute(x, box, style, params, rc)
    fl, El, Wl, nl, rhol = oracle.forces(x, box, style, params, rc, skin=skin)
    assert nb == nl
    assert El == pytest.approx(Eb, rel=1e-13)
    assert np.allclose(Wl, Wb, rtol=1e-12, atol=1e-12 * np.abs(Wb).max())
    assert np.abs(fl - fb).max() < 1e-12 * np.abs(fb).max()
    if rhob is not None:
        assert np.allclose(rhol, rhob, rtol=1e-13)


def test_neighbor_set_matches_brute_force():
    """Full list == both orientations of the brute-force pair set; symmetric; unwrapped input is fine."""
    w = wl.make(1, n_override=6)
    x = wl.perturbed(w, 0.2, seed=5)
    rl = 2.8
    pi, pj = oracle.pairs_brute(x, w.box, rl)
    brute = set(zip(pi.tolist(), pj.tolist()))
    shift = np.array([w.box[0], -2 * w.box[1], 0.0])               # same atoms, other periodic images
    for xs in (x, x + shift * (np.arange(len(x)) % 2)[:, None]):
        start, idx = oracle.NeighborList(xs, w.box, rl).csr()
        full = set()
        for i in range(len(x)):
            for j in idx[start[i]:start[i + 1]]:
                assert j != i
                full.add((i, int(j)))
        assert len(full) == start[-1]                              # no duplicates
        assert full == brute | {(j, i) for (i, j) in brute}
    cnt, nb = oracle.neighbors_sample(x, w.box, rl, [0, 17, 500])
    for s, i in enumerate([0, 17, 500]):
        assert list(nb[s, :cnt[s]]) == sorted(j for (a, j) in full if a == i)


def test_sampled_forces_match_brute_force():
    for style in (oracle.PAIR_LJ, oracle.PAIR_EAM):
        x, box, params, rc = _small_system(style)
        fb, Eb, _, _, _ = oracle.forces_brute(x, box, style, params, rc)
        ids = np.arange(0, x.shape[0], 29)
        fs, es = oracle.forces_sample(x, box, style, params, rc, ids)
        assert np.abs(fs - fb[ids]).max() < 1e-12 * np.abs(fb).max()
        f_all, e_all = oracle.forces_sample(x, box, style, params, rc, np.arange(x.shape[0]))
        assert e_all.sum() == pytest.approx(Eb, rel=1e-12)


def test_box_smaller_than_three_cells_is_refused():
    x, box = wl.fcc_lattice(4, wl.LJ_A)                            # L = 6.72 < 3 * 2.8
    with pytest.raises(ValueError):
        oracle.NeighborList(x, box, 2.8)
