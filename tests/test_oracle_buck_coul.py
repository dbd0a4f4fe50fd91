"""Pins of the oracle's Buckingham + cutoff-Coulomb pair style (App. A: the
"silicate (cutoff)" workload, LAMMPS style buck/coul/cut) against things other than itself.

    u_ab(r) = A_ab exp(-r/rho_ab) - C_ab / r^6 + k q_a q_b / r,   r^2 < rc^2, plain truncation.

Each of the three terms is pinned separately by a reduction to something already pinned or to a closed form:
  * exponential term  == the EAM pair function phi with the embedding switched off (B = 0): pinned by the EAM lattice
    sums and two-atom closed forms of test_oracle_pins.py;
  * dispersion term   == the difference of two LJ systems that share the repulsive coefficient (4 eps s^12):
    LJ(eps', s') - LJ(eps, s) = -4 eps s^6 (g^6 - 1) / r^6 for eps' = eps g^12, s' = s / g -- the LJ function is pinned
    by exact decimals;
  * Coulomb term      == k q_a q_b / r exact decimals for two ions, and the cutoff lattice energy of rock salt by direct
    lattice-vector enumeration (a different algorithm from the oracle's minimum-image loops);
and the sum by finite differences of the energy (forces, virial), Newton's third law, the strict cutoff, the symmetry
of the type table and the equality of the O(N^2) and the list route on a two-species system.
"""
import numpy as np
import pytest

import oracle

K = 14.399645   # eV A / e^2 (LAMMPS metal units qqr2e)
BOX = np.array([24.0, 24.0, 24.0])


def table(nt, A=0.0, rho=1.0, C=0.0):
    c = np.zeros((nt, nt, 3))
    c[..., 0], c[..., 1], c[..., 2] = A, rho, C
    return c


def params(types, q, coef, k=K):
    return dict(k=k, types=np.asarray(types, np.int32), q=np.asarray(q, float), coef=coef)


def two_ions(r, axis=0):
    x = np.array([[5.0, 6.0, 7.0], [5.0, 6.0, 7.0]])
    x[1, axis] += r
    return x


def silicate_like(n=4, seed=7, amp=0.15):
    """Rock-salt arrangement of two species (types alternate with the parity of ix+iy+iz), jittered."""
    a = 2.3
    g = np.arange(n)
    ix, iy, iz = np.meshgrid(g, g, g, indexing="ij")
    x = np.stack([ix, iy, iz], -1).reshape(-1, 3) * a
    types = ((ix + iy + iz) % 2).reshape(-1).astype(np.int32)
    rng = np.random.default_rng(seed)
    x = x + rng.uniform(-amp, amp, x.shape)
    box = np.array([n * a] * 3)
    coef = np.zeros((2, 2, 3))
    coef[0, 0] = (1388.77, 0.3623, 175.0)     # stated synthetic parameters (O-O-like)
    coef[1, 1] = (0.0, 1.0, 0.0)              # cation-cation: Coulomb only
    coef[0, 1] = coef[1, 0] = (18003.76, 0.2052, 133.54)
    return x, box, types, [-1.2, 2.4 / 2.0], coef


# ---- the three terms, one at a time -------------------------------------------------------------------

@pytest.mark.parametrize("axis", [0, 1, 2])
def test_coulomb_two_ions_exact_decimals(axis):
    # k q1 q2 / r with k = 14.399645: r = 2, q = +1, -1 -> -7.1998225 eV; force magnitude k/r^2 = 3.59991125 eV/A, attractive
    P = params([0, 1], [1.0, -1.0], table(2))
    f, E, W, n, _ = oracle.forces_brute(two_ions(2.0, axis), BOX, oracle.PAIR_BUCK_COUL, P, 8.0)
    assert n == 1 and E == pytest.approx(-7.1998225, abs=1e-13)
    assert f[1, axis] == pytest.approx(-3.59991125, abs=1e-13) and f[0, axis] == pytest.approx(3.59991125, abs=1e-13)
    assert np.abs(np.delete(f, axis, 1)).max() == 0.0
    # like charges repel; q = 2.4, -1.2 at r = 1.6: -25.919361 * ... = k * (-2.88) / 1.6
    P = params([0, 1], [2.4, -1.2], table(2))
    E = oracle.forces_brute(two_ions(1.6, axis), BOX, oracle.PAIR_BUCK_COUL, P, 8.0)[1]
    assert E == pytest.approx(-25.919361, abs=1e-12)
    P = params([0, 0], [1.5], table(1))
    f, E = oracle.forces_brute(two_ions(3.0, axis), BOX, oracle.PAIR_BUCK_COUL, P, 8.0)[:2]
    assert E == pytest.approx(10.79973375, abs=1e-12) and f[1, axis] > 0 > f[0, axis]


def test_exponential_term_equals_eam_pair_function_without_embedding():
    x, box, types, q, _ = silicate_like()
    A, rho, rc = 1388.77, 0.3623, 5.5
    P = params(np.zeros(len(x), np.int32), [0.0], table(1, A=A, rho=rho))
    fb, Eb, Wb, nb, _ = oracle.forces_brute(x, box, oracle.PAIR_BUCK_COUL, P, rc)
    # phi(r) = A' exp(-p (r/r0 - 1)) with p / r0 = 1 / rho and A' = A exp(-r0 / rho); B = 0 switches the embedding off
    r0 = 2.0
    fe, Ee, We, ne, _ = oracle.forces_brute(x, box, oracle.PAIR_EAM, (A * np.exp(-r0 / rho), r0 / rho, 0.0, 1.0, r0), rc)
    assert nb == ne and Eb == pytest.approx(Ee, rel=1e-13)
    assert np.abs(fb - fe).max() < 1e-12 * np.abs(fe).max() and np.allclose(Wb, We, rtol=1e-12, atol=1e-12)


def test_dispersion_term_equals_difference_of_two_lj_systems():
    x, box, types, q, _ = silicate_like()
    eps, s, g, rc = 0.7, 1.9, 1.25, 5.5
    C = 4.0 * eps * s ** 6 * (g ** 6 - 1.0)
    P = params(np.zeros(len(x), np.int32), [0.0], table(1, A=0.0, rho=1.0, C=C))
    fb, Eb, Wb = oracle.forces_brute(x, box, oracle.PAIR_BUCK_COUL, P, rc)[:3]
    f1, E1, W1 = oracle.forces_brute(x, box, oracle.PAIR_LJ, (eps, s), rc)[:3]
    f2, E2, W2 = oracle.forces_brute(x, box, oracle.PAIR_LJ, (eps * g ** 12, s / g), rc)[:3]
    # the two LJ systems have the same 4 eps s^12: their difference is the pure -C/r^6 term (up to cancellation rounding)
    scale = np.abs(f1).max()
    assert Eb == pytest.approx(E2 - E1, abs=1e-10 * abs(E1))
    assert np.abs(fb - (f2 - f1)).max() < 1e-10 * scale and np.allclose(Wb, W2 - W1, atol=1e-9 * abs(W1).max())


def test_rock_salt_cutoff_coulomb_energy_by_lattice_vector_enumeration():
    n, a, rc, q = 6, 2.0, 5.7, 0.9
    g = np.arange(n)
    ix, iy, iz = np.meshgrid(g, g, g, indexing="ij")
    x = np.stack([ix, iy, iz], -1).reshape(-1, 3) * a
    types = ((ix + iy + iz) % 2).reshape(-1)
    P = params(types, [q, -q], table(2))
    f, E, W, npairs, _ = oracle.forces_brute(x, np.array([n * a] * 3), oracle.PAIR_BUCK_COUL, P, rc)
    # independent: every site sees the same shells; sum over integer lattice vectors inside the cutoff sphere
    m = int(rc / a) + 1
    e_site, count = 0.0, 0
    for i in range(-m, m + 1):
        for j in range(-m, m + 1):
            for k in range(-m, m + 1):
                r = a * (i * i + j * j + k * k) ** 0.5
                if 0.0 < r < rc:
                    e_site += (-1.0) ** (i + j + k) * K * q * q / r
                    count += 1
    assert npairs == len(x) * count // 2
    assert E == pytest.approx(0.5 * len(x) * e_site, rel=1e-12)
    assert np.abs(f).max() < 1e-10          # every site is a centre of symmetry


# ---- the whole function ---------------------------------------------------------------------------------

def test_forces_and_virial_are_energy_derivatives_two_species():
    x, box, types, q, coef = silicate_like()
    rc = 5.5
    P = params(types, q, coef)
    f, E, W = oracle.forces_brute(x, box, oracle.PAIR_BUCK_COUL, P, rc)[:3]
    pi, pj, r2 = oracle.pairs_brute(x, box, rc + 0.01, with_r2=True)
    assert np.abs(np.sqrt(r2) - rc).min() > 1e-4            # no pair crosses the cutoff under the displacements below
    h = 1e-5
    rng = np.random.default_rng(3)
    for i in rng.choice(len(x), 6, replace=False):
        for a in range(3):
            xp, xm = x.copy(), x.copy()
            xp[i, a] += h; xm[i, a] -= h
            Ep = oracle.forces_brute(xp, box, oracle.PAIR_BUCK_COUL, P, rc)[1]
            Em = oracle.forces_brute(xm, box, oracle.PAIR_BUCK_COUL, P, rc)[1]
            assert f[i, a] == pytest.approx(-(Ep - Em) / (2 * h), rel=2e-7, abs=1e-6)
    # tr W = -dE/d ln(scale), each diagonal component by stretching one axis
    for a in range(3):
        sp = np.ones(3); sp[a] += h
        sm = np.ones(3); sm[a] -= h
        Ep = oracle.forces_brute(x * sp, box * sp, oracle.PAIR_BUCK_COUL, P, rc)[1]
        Em = oracle.forces_brute(x * sm, box * sm, oracle.PAIR_BUCK_COUL, P, rc)[1]
        assert W[a] == pytest.approx(-(Ep - Em) / (2 * h), rel=1e-6, abs=1e-5)
    assert np.abs(f.sum(0)).max() < 1e-10 * np.abs(f).max() * len(x)          # Newton's third law


def test_cutoff_is_strict_and_type_table_is_used_per_pair():
    coef = np.zeros((2, 2, 3))
    coef[0, 0] = (100.0, 0.5, 3.0); coef[1, 1] = (50.0, 0.4, 1.0); coef[0, 1] = coef[1, 0] = (75.0, 0.45, 2.0)
    E = {}
    for ta, tb in [(0, 0), (0, 1), (1, 0), (1, 1)]:
        P = params([ta, tb], [0.3, -0.6], coef)
        E[ta, tb] = oracle.forces_brute(two_ions(2.0), BOX, oracle.PAIR_BUCK_COUL, P, 3.0)[1]
        assert oracle.forces_brute(two_ions(3.0), BOX, oracle.PAIR_BUCK_COUL, P, 3.0)[3] == 0          # r == rc is outside
        assert oracle.forces_brute(two_ions(2.999), BOX, oracle.PAIR_BUCK_COUL, P, 3.0)[3] == 1
    assert E[0, 1] == E[1, 0] and len({E[0, 0], E[0, 1], E[1, 1]}) == 3
    with pytest.raises(ValueError):
        bad = coef.copy(); bad[0, 1, 0] = 1.0
        oracle.forces_brute(two_ions(2.0), BOX, oracle.PAIR_BUCK_COUL, params([0, 1], [0.3, -0.6], bad), 3.0)


def test_list_route_and_sampled_scans_match_brute_force_two_species():
    x, box, types, q, coef = silicate_like(n=8)
    rc, skin = 5.5, 0.6
    P = params(types, q, coef)
    fb, Eb, Wb, nb, _ = oracle.forces_brute(x, box, oracle.PAIR_BUCK_COUL, P, rc)
    fl, El, Wl, nl, _ = oracle.forces(x, box, oracle.PAIR_BUCK_COUL, P, rc, skin=skin)
    assert nl == nb and El == pytest.approx(Eb, rel=1e-12)
    assert np.abs(fl - fb).max() < 1e-11 * np.abs(fb).max() and np.allclose(Wl, Wb, rtol=1e-10, atol=1e-9)
    ids = np.array([0, 17, 255, len(x) - 1])
    fs, es = oracle.forces_sample(x, box, oracle.PAIR_BUCK_COUL, P, rc, ids)
    assert np.abs(fs - fb[ids]).max() < 1e-11 * np.abs(fb).max()
