"""Parity of the CUDA path (through the C ABI) with the CPU oracle, element by element, on the same
seeded inputs.  Tolerances (BASELINE.json north_star):

  pair sets     identical, pairs within 1e-9 sigma of rc+skin excluded
  fp64 forces   max |dF| <= 1e-12 * max(|F_i|, F_rms) per atom; energy/virial 1e-12 relative
  mixed forces  relative RMS sqrt(sum|dF|^2 / sum|F|^2) <= 1e-5; energy 1e-6 relative
"""
import numpy as np
import pytest

import oracle
from paper_1009_4330_b200 import workloads as wl

pytestmark = pytest.mark.gpu

md = None


@pytest.fixture(scope="module", autouse=True)
def _load_md():
    global md
    from paper_1009_4330_b200 import md as _md
    md = _md
    yield


def _rel_rms(f, ref):
    return float(np.sqrt(((f - ref) ** 2).sum() / (ref ** 2).sum()))


def _fp64_force_err(f, ref):
    mag = np.sqrt((ref ** 2).sum(axis=1))
    floor = np.sqrt((mag ** 2).mean())
    return float((np.abs(f - ref).max(axis=1) / np.maximum(mag, floor)).max())


def _system(cfg, n, amp, precision, kernel, list_kind=0, seed=7):
    w = wl.make(cfg, n_override=n)
    x = wl.perturbed(w, amp, seed=seed)
    s = md.from_workload(w, precision=precision, list_kind=list_kind, kernel=kernel, x=x)
    return w, x, s


def _oracle_pairs(x, box, rl, band=1e-9):
    pi, pj, r2 = oracle.pairs_brute(x, box, rl + 10 * band, with_r2=True)
    r = np.sqrt(r2)
    sure = r < rl - band
    fuzzy = ~sure
    return (set(zip(pi[sure].tolist(), pj[sure].tolist())),
            set(zip(pi[fuzzy].tolist(), pj[fuzzy].tolist())))


def _gpu_rows(s, N, stride):
    nn = np.zeros(N, np.int32)
    nb = np.full(N * stride, -1, np.int32)
    s.md_get_neighbors(nn, nb, stride)
    assert nn.max() <= stride
    return nn, nb.reshape(N, stride)


# ---- neighbor sets -----------------------------------------------------------------------------------------

@pytest.mark.parametrize("cfg,n,amp,kernel", [
    (1, 6, 0.15, 1), (1, 7, 0.15, 2), (1, 10, 0.15, 3), (4, 5, 0.2, 1), (4, 7, 0.2, 2),
])
def test_full_list_pair_set_matches_brute_force(cfg, n, amp, kernel):
    w, x, s = _system(cfg, n, amp, md.MD_FP64, kernel)
    s.md_build_neighbors()
    rl = w.rc + w.skin
    sure, fuzzy = _oracle_pairs(x, w.box, rl)
    nn, nb = _gpu_rows(s, w.natoms, 1024 if cfg != 4 else 256)
    got = set()
    for i in range(w.natoms):
        row = nb[i, :nn[i]]
        assert len(set(row.tolist())) == nn[i], "duplicate neighbor in a row"
        got.update((i, int(j)) for j in row)
    assert all((j, i) in got for (i, j) in got), "full list must be symmetric"
    und = {(min(i, j), max(i, j)) for (i, j) in got}
    assert sure <= und and und <= (sure | fuzzy)
    assert len(got) == 2 * len(und)
    st = s.md_get_stats()
    assert st["nbuilds"] >= 1 and st["max_neighbors"] == nn.max()
    assert st["mean_neighbors"] == pytest.approx(nn.mean(), rel=1e-12)


@pytest.mark.parametrize("precision", [0, 1])
@pytest.mark.parametrize("kernel,list_kind", [(1, 0), (2, 0), (1, 1)])
def test_pairs_at_the_list_radius_are_decided_in_fp64(kernel, list_kind, precision):
    """The build's distance test runs in fp32 and accepts everything up to a guard band beyond rl (the stored rows
    are a superset); the pair set the library reports is decided in fp64.  Dimers are planted at r = rl (1 +- d) with d from 1e-5 down to 3e-9 (far inside the fp32 band,
    outside the 1e-9 exclusion of the comparison), in random orientations, all over a periodic box, so that the
    partner sits in any of the 27 stencil cells and across the periodic boundary."""
    rc, skin = 2.5, 0.3
    rl = rc + skin
    box = np.array([31.0, 29.0, 33.0])
    nd = 600
    ids = np.arange(nd, dtype=np.uint64)
    centre = np.stack([wl.uniform01(11, ids, c) for c in range(3)], axis=1) * box
    u = np.stack([wl.gaussian(11, ids, 3 + c) for c in range(3)], axis=1)
    u /= np.linalg.norm(u, axis=1)[:, None]
    deltas = np.array([1e-5, 1e-6, 1e-7, 1e-8, 3e-9])
    d = deltas[np.arange(nd) % 5] * np.where((np.arange(nd) // 5) % 2 == 0, 1.0, -1.0)
    x = np.concatenate([centre, centre + u * (rl * (1.0 + d))[:, None]])      # partner may lie outside the box
    N = 2 * nd
    s = md.System(box, N, np.zeros(N, np.int32), np.array([1.0]))
    s.md_set_precision(precision)
    s.md_set_neighbor(list_kind, kernel)
    s.md_set_pair(md.MD_PAIR_LJ126, (1.0, 1.0), rc, skin)
    s.md_set_positions(x)
    s.md_build_neighbors()
    nn, nb = _gpu_rows(s, N, 64)
    got = {(min(i, int(j)), max(i, int(j))) for i in range(N) for j in nb[i, :nn[i]]}
    sure, fuzzy = _oracle_pairs(x, box, rl)
    assert sure <= got and got <= (sure | fuzzy)
    # the planted dimers themselves: inside iff d < 0, judged from the fp64 coordinates actually passed in
    xw = x - np.floor(x / box) * box
    dd = xw[:nd] - xw[nd:]
    dd -= box * np.round(dd / box)
    r = np.sqrt((dd ** 2).sum(axis=1))
    decided = np.abs(r - rl) > 1e-9
    assert decided.sum() > 0.9 * nd
    for k in np.nonzero(decided)[0]:
        assert ((k, nd + k) in got) == (r[k] < rl), (k, r[k] - rl)
    s.close()


@pytest.mark.parametrize("cfg,n,amp,kernel,list_kind,precision", [
    (1, 6, 0.15, 1, 0, 0), (2, 8, 0.15, 1, 0, 1), (1, 7, 0.15, 2, 0, 1), (4, 6, 0.2, 1, 0, 1), (1, 7, 0.15, 1, 1, 1),
])
def test_stored_rows_are_a_tight_superset(cfg, n, amp, kernel, list_kind, precision):
    """What the build kernel itself writes (md_get_neighbor_rows): one row per pair of consecutive atoms of a cell,
    holding the union of the two atoms' neighbors without the two atoms themselves.  Every row must contain all
    fp64 neighbors of both atoms (nothing missed) and nothing beyond the fp32 guard band around rl (no junk);
    for a half list the same with 'neighbors' = the partners the exact export assigns to the two atoms."""
    w, x, s = _system(cfg, n, amp, precision, kernel, list_kind)
    s.md_build_neighbors()
    N = w.natoms
    rl = w.rc + w.skin
    st = s.md_get_stats()
    stride = int(st["max_row"]) + 8
    owner = np.zeros(N, np.int32); nrow = np.zeros(N, np.int32); ent = np.full(N * stride, -1, np.int32)
    s.md_get_neighbor_rows(owner, nrow, ent, stride)
    ent = ent.reshape(N, stride)
    nn, nb = _gpu_rows(s, N, 1024 if cfg != 4 else 256)
    exact = [set(nb[i, :nn[i]].tolist()) for i in range(N)]
    pi, pj, _ = oracle.pairs_brute(x, w.box, rl * (1.0 + 2e-5), with_r2=True)
    loose = [set() for _ in range(N)]
    for a, b in zip(pi.tolist(), pj.tolist()):
        loose[a].add(b); loose[b].add(a)
    firsts = np.nonzero(owner == np.arange(N))[0]
    seconds = np.nonzero(owner != np.arange(N))[0]
    assert len(firsts) + len(seconds) == N and len(seconds) <= len(firsts)
    assert np.all(owner[owner[seconds]] == owner[seconds]) and np.all(nrow[seconds] == 0)
    assert len(set(owner[seconds].tolist())) == len(seconds), "an atom is the partner of two first atoms"
    partner = {int(owner[j]): int(j) for j in seconds}
    assert nrow[firsts].max() == st["max_row"]
    assert nrow[firsts].sum() / (0.5 * N) == pytest.approx(st["mean_row"], rel=1e-12)
    total_exact = 0
    for i0 in firsts.tolist():
        row = ent[i0, :nrow[i0]].tolist()
        have = set(row)
        assert len(have) == len(row), "duplicate entry in a stored row"
        pair = {i0} | ({partner[i0]} if i0 in partner else set())
        assert not (have & pair), "a pair's own atoms must not be entries of its row"
        need = set().union(*(exact[a] for a in pair)) - pair
        allow = set().union(*(loose[a] for a in pair))
        assert need <= have <= allow
        total_exact += sum(len(exact[a]) for a in pair)
    assert total_exact == nn.sum()
    # the union costs less than 1.6 single rows in these dense systems (the point of pairing spatial neighbours)
    if list_kind == 0:
        assert st["mean_row"] < 1.6 * st["mean_neighbors"]
    s.close()


def test_half_list_holds_each_pair_once():
    w, x, s = _system(1, 7, 0.15, md.MD_FP64, md.MD_KERNEL_TPA, list_kind=md.MD_LIST_HALF)
    s.md_build_neighbors()
    sure, fuzzy = _oracle_pairs(x, w.box, w.rc + w.skin)
    nn, nb = _gpu_rows(s, w.natoms, 256)
    got = [(i, int(j)) for i in range(w.natoms) for j in nb[i, :nn[i]]]
    und = {(min(i, j), max(i, j)) for (i, j) in got}
    assert len(und) == len(got), "a pair appears in both rows or twice"
    assert sure <= und and und <= (sure | fuzzy)


# ---- forces, energy, virial: small boxes, every kernel variant, against the O(N^2) definition --------------

VARIANTS = [("tpa", 1, 0), ("subwarp2", 6, 0), ("subwarp4", 5, 0), ("subwarp8", 2, 0), ("warp", 3, 0), ("cell", 4, 0), ("half", 1, 1)]


@pytest.mark.parametrize("name,kernel,list_kind", VARIANTS)
@pytest.mark.parametrize("cfg,n,amp", [(1, 6, 0.12), (1, 9, 0.12), (4, 5, 0.25), (4, 8, 0.25)])
def test_fp64_forces_energy_virial(cfg, n, amp, name, kernel, list_kind):
    w, x, s = _system(cfg, n, amp, md.MD_FP64, kernel, list_kind)
    fo, Eo, Wo, npairs, _ = oracle.forces_brute(x, w.box, w.style, w.params, w.rc)
    f = np.zeros((w.natoms, 3))
    E, W = s.md_compute_forces(f, energy=True, virial=True)
    assert _fp64_force_err(f, fo) < 1e-12
    assert E == pytest.approx(Eo, rel=1e-12)
    assert np.abs(W - Wo).max() < 1e-12 * np.abs(Wo).max()
    assert np.abs(f.sum(axis=0)).max() < 1e-10 * np.abs(f).sum()
    g = np.zeros((w.natoms, 3))
    s.md_get_forces(g)
    assert np.array_equal(f, g)


@pytest.mark.parametrize("name,kernel,list_kind", VARIANTS)
@pytest.mark.parametrize("cfg,n,amp", [(2, 8, 0.12), (4, 8, 0.25)])
def test_mixed_forces_energy_virial(cfg, n, amp, name, kernel, list_kind):
    w, x, s = _system(cfg, n, amp, md.MD_MIXED, kernel, list_kind)
    fo, Eo, Wo, _, _ = oracle.forces_brute(x, w.box, w.style, w.params, w.rc)
    f = np.zeros((w.natoms, 3))
    E, W = s.md_compute_forces(f, energy=True, virial=True)
    assert _rel_rms(f, fo) < 1e-5
    assert abs(E - Eo) < 1e-6 * abs(Eo)
    assert np.abs(W - Wo).max() < 1e-5 * np.abs(Wo).max()


def test_variants_agree_bitwise_on_repeat_and_closely_with_each_other():
    """Same input twice gives the same bits (deterministic order); variants differ only in summation order."""
    res = {}
    for name, kernel, list_kind in VARIANTS:
        w, x, s = _system(1, 8, 0.12, md.MD_FP64, kernel, list_kind)
        f1, f2 = np.zeros((w.natoms, 3)), np.zeros((w.natoms, 3))
        s.md_compute_forces(f1)
        s.md_set_positions(x)
        s.md_compute_forces(f2)
        if name != "half":   # atomics: order not fixed
            assert np.array_equal(f1, f2)
        res[name] = f1
    for name in res:
        assert _fp64_force_err(res[name], res["tpa"]) < 1e-12


def test_two_atoms_analytic_through_the_api():
    box = np.array([10.0, 10.0, 10.0])
    rmin = 2.0 ** (1.0 / 6.0)
    for prec, tol in [(md.MD_FP64, 1e-13), (md.MD_MIXED, 2e-6)]:
        for r, Eexp, Fexp in [(1.0, 0.0, 24.0), (rmin, -1.0, 0.0), (2.4, None, None)]:
            x = np.array([[9.7, 5.0, 5.0], [9.7 + r - 10.0, 5.0, 5.0]])   # across the periodic face
            s = md.System(box, 2, np.zeros(2, np.int32), np.array([1.0]))
            s.md_set_precision(prec)
            s.md_set_pair(md.MD_PAIR_LJ126, (1.0, 1.0), 2.5, 0.3)
            s.md_set_positions(x)
            f = np.zeros((2, 3))
            E, W = s.md_compute_forces(f, energy=True, virial=True)
            if Eexp is None:
                Eexp = 4.0 * (r ** -12 - r ** -6)
                Fexp = 24.0 * (2.0 * r ** -12 - r ** -6) / r
            assert abs(E - Eexp) < tol * max(1.0, abs(Eexp))
            assert abs(f[0, 0] - (-Fexp)) < tol * 24.0 and abs(f[1, 0] - Fexp) < tol * 24.0
            assert np.abs(f[:, 1:]).max() == 0.0
            assert abs(W[0] - r * Fexp) < tol * 24.0
            s.close()


def test_caller_order_and_permutation_invariance():
    """cfg 5 shuffles atom order: results in caller order equal the unshuffled run mapped through the
    permutation, to rounding (the internal spatial sort is invisible)."""
    w = wl.make(5, n_override=8)
    x = wl.perturbed(w, 0.1, seed=3)
    s = md.from_workload(w, precision=md.MD_FP64, x=x)
    f = np.zeros((w.natoms, 3))
    s.md_compute_forces(f)
    order = np.argsort(wl.permutation(w.seed, w.natoms))      # undo the shuffle
    w2 = wl.make(5, n_override=8)
    w2.x, w2.v = x[order].copy(), w.v[order].copy()
    s2 = md.from_workload(w2, precision=md.MD_FP64)
    f2 = np.zeros((w.natoms, 3))
    s2.md_compute_forces(f2)
    assert _fp64_force_err(f, f2[np.argsort(order)]) < 1e-12
    xb = np.zeros((w.natoms, 3))
    s.md_get_positions(xb)
    d = xb - x
    d -= w.box * np.round(d / w.box)
    assert np.abs(d).max() < 1e-13


# ---- time stepping ----------------------------------------------------------------------------------------

def _minimg(d, box):
    return d - box * np.round(d / box)


def test_cfg1_trajectory_fp64_100_steps():
    """Config 1 as stated: 4,000 atoms, fp64, 100 NVE steps; pointwise against the oracle's trajectory
    (0.5 tau: rounding differences grow by < 1e4, so 1e-9 is a real bound)."""
    w = wl.make(1)
    s = md.from_workload(w)
    s.md_run(w.nsteps, w.dt)
    x, v, f = (np.zeros((w.natoms, 3)) for _ in range(3))
    s.md_get_positions(x); s.md_get_velocities(v); s.md_get_forces(f)
    ref = oracle.run_nve(w.x, w.v, w.box, np.ones(w.natoms), w.style, w.params, w.rc, w.skin, w.dt, w.nsteps)
    assert np.abs(_minimg(x - ref["x"], w.box)).max() < 1e-9
    assert np.abs(v - ref["v"]).max() < 1e-8
    assert _fp64_force_err(f, ref["f"]) < 1e-7
    st = s.md_get_stats()
    assert st["nsteps_total"] == w.nsteps
    assert abs(st["nbuilds"] - ref["nbuild"]) <= 1
    ke = 0.5 * (ref["v"] ** 2).sum()
    assert st["kinetic_energy"] == pytest.approx(ke, rel=1e-9)
    # same-input snapshot: the oracle recomputes forces from the GPU's own final positions
    fo = oracle.forces(x, w.box, w.style, w.params, w.rc)[0]
    assert _fp64_force_err(f, fo) < 1e-12


@pytest.mark.parametrize("kernel,list_kind", [(1, 0), (2, 0), (3, 0), (4, 0), (5, 0), (1, 1)])
def test_run_in_pieces_equals_run_at_once_and_snapshots_match(kernel, list_kind):
    w = wl.make(1, n_override=7)
    a = md.from_workload(w, precision=md.MD_FP64, kernel=kernel, list_kind=list_kind)
    b = md.from_workload(w, precision=md.MD_FP64, kernel=kernel, list_kind=list_kind)
    a.md_run(60, w.dt)
    for _ in range(3):
        b.md_run(20, w.dt)
    xa, xb, f = (np.zeros((w.natoms, 3)) for _ in range(3))
    a.md_get_positions(xa); b.md_get_positions(xb)
    assert np.abs(_minimg(xa - xb, w.box)).max() < 1e-10
    a.md_get_forces(f)
    fo = oracle.forces(xa, w.box, w.style, w.params, w.rc)[0]
    assert _fp64_force_err(f, fo) < 1e-12
    # list validity: every pair inside rc is in the list the run left behind
    nn, nb = _gpu_rows(a, w.natoms, 256)
    pi, pj = oracle.pairs_brute(xa, w.box, w.rc - 1e-9)
    have = {(i, int(j)) for i in range(w.natoms) for j in nb[i, :nn[i]]}
    if list_kind == 0:
        assert all((i, j) in have and (j, i) in have for i, j in zip(pi.tolist(), pj.tolist()))
    else:
        assert all(((i, j) in have) != ((j, i) in have) for i, j in zip(pi.tolist(), pj.tolist()))


def test_mixed_run_conserves_energy_and_momentum_cfg2_small():
    """NVE drift is judged on the SHIFTED energy E - npairs u(rc) (reading s2: lj/cut is plainly truncated, so
    every pair crossing rc jumps E by u(rc) = -0.0163; the melting lattice gains ~2000 in-range pairs)."""
    w = wl.make(2, n_override=10)
    urc = 4.0 * (w.rc ** -12 - w.rc ** -6)
    s = md.from_workload(w)
    E0, _ = s.md_compute_forces(energy=True)
    ke0 = s.md_get_stats()["kinetic_energy"]
    np0 = oracle.forces(w.x, w.box, w.style, w.params, w.rc)[3]
    s.md_run(200, w.dt)
    E1, _ = s.md_compute_forces(energy=True)
    ke1 = s.md_get_stats()["kinetic_energy"]
    v = np.zeros((w.natoms, 3))
    s.md_get_velocities(v)
    # fp32 pair terms are rounded differently in the tiles of i and of j, so Newton's third law holds only to
    # fp32 rounding with a full list: the net momentum random-walks at ~1e-8 per atom per 100 steps
    assert np.abs(v.sum(axis=0)).max() < 1e-6 * w.natoms
    x = np.zeros((w.natoms, 3))
    s.md_get_positions(x)
    fo, Eo, _, np1, _ = oracle.forces(x, w.box, w.style, w.params, w.rc)
    drift = (E1 - np1 * urc + ke1) - (E0 - np0 * urc + ke0)
    assert abs(drift) < 1e-4 * w.natoms, drift          # the fp64 oracle drifts by -0.09 on this input
    f = np.zeros((w.natoms, 3))
    s.md_get_forces(f)
    assert _rel_rms(f, fo) < 1e-5 and abs(E1 - Eo) < 1e-6 * abs(Eo)


@pytest.mark.parametrize("precision", [0, 1])
@pytest.mark.parametrize("kernel", [1, 5, 2, 3])
def test_long_lived_list_is_balanced_and_stays_correct(kernel, precision):
    """A cold solid keeps its list for hundreds of steps; after 48 steps md_run permutes the rows for conflict-free
    shared-memory gathers (a pure reordering within each stored row).  Forces, energy and the stored rows (as sets)
    must not change."""
    w = wl.make(4, n_override=6)
    s = md.from_workload(w, precision=precision, kernel=kernel)
    N = w.natoms

    def stored_rows():
        owner = np.zeros(N, np.int32); nrow = np.zeros(N, np.int32); ent = np.full(N * 192, -1, np.int32)
        s.md_get_neighbor_rows(owner, nrow, ent, 192)
        return owner, nrow, ent.reshape(N, 192)

    s.md_run(40, w.dt)
    assert s.md_get_stats()["list_balanced"] == 0
    o0, n0, e0 = stored_rows()
    s.md_run(40, w.dt)
    st = s.md_get_stats()
    assert st["list_balanced"] == 1 and st["nbuilds"] == 1
    o1, n1, e1 = stored_rows()
    assert np.array_equal(o0, o1) and np.array_equal(n0, n1)
    for i in range(N):
        assert sorted(e0[i, :n0[i]].tolist()) == sorted(e1[i, :n1[i]].tolist())
    x, f = np.zeros((w.natoms, 3)), np.zeros((w.natoms, 3))
    s.md_get_positions(x)
    E, W = s.md_compute_forces(f, energy=True, virial=True)
    fo, Eo, Wo, _, _ = oracle.forces(x, w.box, w.style, w.params, w.rc)
    if precision == md.MD_FP64:
        assert _fp64_force_err(f, fo) < 1e-12 and abs(E - Eo) < 1e-12 * abs(Eo)
    else:
        assert _rel_rms(f, fo) < 1e-5 and abs(E - Eo) < 1e-6 * abs(Eo)
    s.close()


def test_eam_metal_units_run_matches_oracle():
    w = wl.make(4, n_override=6)
    s = md.from_workload(w, precision=md.MD_FP64)
    s.md_run(40, w.dt)
    x, v = np.zeros((w.natoms, 3)), np.zeros((w.natoms, 3))
    s.md_get_positions(x); s.md_get_velocities(v)
    ref = oracle.run_nve(w.x, w.v, w.box, np.full(w.natoms, w.mass[0]), w.style, w.params, w.rc, w.skin, w.dt, 40,
                         ftm2v=w.ftm2v, mvv2e=w.mvv2e)
    assert np.abs(_minimg(x - ref["x"], w.box)).max() < 1e-10
    assert np.abs(v - ref["v"]).max() < 1e-9
    ke = 0.5 * w.mvv2e * w.mass[0] * (ref["v"] ** 2).sum()
    assert s.md_get_stats()["kinetic_energy"] == pytest.approx(ke, rel=1e-10)


@pytest.mark.parametrize("cfg,n,nsteps", [(1, 7, 80), (4, 6, 40)])
def test_half_list_run_matches_oracle_trajectory(cfg, n, nsteps):
    """Half list (Newton's third law) through md_run: the batched three-launch time step (kick+drift |
    scatter forces | kick) with the device-side stale flag must rebuild at the oracle's steps (+-1) and follow
    its trajectory; LJ (hot liquid: several rebuilds inside the run) and two-pass EAM."""
    w = wl.make(cfg, n_override=n)
    s = md.from_workload(w, precision=md.MD_FP64, kernel=md.MD_KERNEL_TPA, list_kind=md.MD_LIST_HALF)
    s.md_run(nsteps, w.dt)
    x, v, f = (np.zeros((w.natoms, 3)) for _ in range(3))
    s.md_get_positions(x); s.md_get_velocities(v); s.md_get_forces(f)
    ref = oracle.run_nve(w.x, w.v, w.box, np.full(w.natoms, w.mass[0]), w.style, w.params, w.rc, w.skin, w.dt, nsteps,
                         ftm2v=w.ftm2v, mvv2e=w.mvv2e)
    assert np.abs(_minimg(x - ref["x"], w.box)).max() < 1e-9
    assert np.abs(v - ref["v"]).max() < 1e-8 * max(1.0, np.abs(ref["v"]).max())
    st = s.md_get_stats()
    assert st["nsteps_total"] == nsteps
    assert abs(st["nbuilds"] - ref["nbuild"]) <= 1
    fo = oracle.forces(x, w.box, w.style, w.params, w.rc)[0]
    assert _fp64_force_err(f, fo) < 1e-11
    s.close()


# ---- Buckingham + cutoff Coulomb, two charged species (App. A) ---------------------

BC_VARIANTS = [("tpa", 1, 0), ("subwarp4", 5, 0), ("warp", 3, 0), ("cell", 4, 0), ("half", 1, 1)]


@pytest.mark.parametrize("name,kernel,list_kind", BC_VARIANTS)
def test_buck_coul_fp64_forces_energy_virial(name, kernel, list_kind):
    w = wl.make(6, n_override=12)                       # 1,728 ions, box = 3 (rc + skin)
    fo, Eo, Wo, npairs, _ = oracle.forces_brute(w.x, w.box, w.style, wl.oracle_params(w), w.rc)
    s = md.from_workload(w, precision=md.MD_FP64, kernel=kernel, list_kind=list_kind)
    f = np.zeros((w.natoms, 3))
    E, W = s.md_compute_forces(f, energy=True, virial=True)
    assert _fp64_force_err(f, fo) < 1e-12
    assert abs(E - Eo) < 1e-12 * abs(Eo) and np.abs(W - Wo).max() < 1e-11 * np.abs(Wo).max()
    s.close()


@pytest.mark.parametrize("name,kernel,list_kind", BC_VARIANTS)
def test_buck_coul_mixed_forces_energy(name, kernel, list_kind):
    w = wl.make(6, n_override=12)
    fo, Eo = oracle.forces_brute(w.x, w.box, w.style, wl.oracle_params(w), w.rc)[:2]
    s = md.from_workload(w, precision=md.MD_MIXED, kernel=kernel, list_kind=list_kind)
    f = np.zeros((w.natoms, 3))
    E, _ = s.md_compute_forces(f, energy=True)
    assert _rel_rms(f, fo) < 1e-5
    assert abs(E - Eo) < 1e-6 * abs(Eo)
    s.close()


def test_buck_coul_type_pairs_and_charges_reach_the_kernel():
    """Two ions of every type combination through the API: the coefficient table is indexed by (t_i, t_j)."""
    box = np.array([40.0, 40.0, 40.0])
    coef = {(0, 0): (100.0, 0.5, 3.0), (0, 1): (75.0, 0.45, 2.0), (1, 1): (50.0, 0.4, 1.0)}
    q = (0.3, -0.6)
    for ta, tb in [(0, 0), (0, 1), (1, 0), (1, 1)]:
        for prec, tol in [(md.MD_FP64, 1e-13), (md.MD_MIXED, 2e-6)]:
            s = md.System(box, 2, np.array([ta, tb], np.int32), np.array([1.0, 2.0]))
            s.md_set_precision(prec)
            s.md_set_pair(md.MD_PAIR_BUCK_COUL, (14.399645,), 6.0, 1.0)
            with pytest.raises(md.MDError) as e:       # coefficients missing
                s.md_set_positions(np.array([[5.0, 5, 5], [7.0, 5, 5]])); s.md_compute_forces()
            assert e.value.code == md.MD_ERR_NOT_READY
            for (a, b), c in coef.items():
                s.md_set_pair_coeff(a, b, c)
            s.md_set_type_charges(q)
            x = np.array([[39.0, 5.0, 5.0], [1.0, 5.0, 5.0]])                     # r = 2 across the periodic face
            s.md_set_positions(x)
            f = np.zeros((2, 3))
            E, _ = s.md_compute_forces(f, energy=True)
            A, rho, C = coef[min(ta, tb), max(ta, tb)]
            P = dict(k=14.399645, types=[ta, tb], q=q, coef=np.array([[coef[0, 0], coef[0, 1]], [coef[0, 1], coef[1, 1]]]))
            fo, Eo = oracle.forces_brute(x, box, oracle.PAIR_BUCK_COUL, P, 6.0)[:2]
            assert abs(E - Eo) < tol * max(1.0, abs(Eo)) and np.abs(f - fo).max() < tol * max(1.0, np.abs(fo).max())
            s.close()


def test_buck_coul_run_matches_oracle_trajectory():
    w = wl.make(6, n_override=12)
    s = md.from_workload(w, precision=md.MD_FP64)
    s.md_run(20, w.dt)
    x, v = np.zeros((w.natoms, 3)), np.zeros((w.natoms, 3))
    s.md_get_positions(x); s.md_get_velocities(v)
    ref = oracle.run_nve(w.x, w.v, w.box, w.mass[w.types], w.style, wl.oracle_params(w), w.rc, w.skin, w.dt, 20,
                         ftm2v=w.ftm2v, mvv2e=w.mvv2e)
    assert np.abs(_minimg(x - ref["x"], w.box)).max() < 1e-9
    assert np.abs(v - ref["v"]).max() < 1e-8 * np.abs(ref["v"]).max()
    s.close()


# ---- SURVEY.md 8(f)-2, second half: tabulated EAM (App. A; reading s26) -------------------------------

@pytest.mark.parametrize("name,kernel,list_kind", [("tpa", 1, 0), ("subwarp4", 5, 0), ("warp", 3, 0), ("cell", 4, 0), ("half", 1, 1)])
@pytest.mark.parametrize("precision", [0, 1])   # MD_FP64, MD_MIXED
def test_tabulated_eam_forces_energy_virial(name, kernel, list_kind, precision):
    w = wl.make_eam_tabulated(6, n_table=1501)
    x = wl.perturbed(w, 0.2)
    fo, Eo, Wo, _, rho_o = oracle.forces_brute(x, w.box, w.style, wl.oracle_params(w), w.rc)
    s = md.from_workload(w, precision=precision, kernel=kernel, list_kind=list_kind, x=x)
    f = np.zeros((w.natoms, 3))
    E, W = s.md_compute_forces(f, energy=True, virial=True)
    if precision == md.MD_FP64:
        assert _fp64_force_err(f, fo) < 1e-11
        assert abs(E - Eo) < 1e-12 * abs(Eo) and np.abs(W - Wo).max() < 1e-10 * np.abs(Wo).max()
    else:
        assert _rel_rms(f, fo) < 1e-5 and abs(E - Eo) < 1e-6 * abs(Eo)
    s.close()


def test_tabulated_eam_run_and_table_checks():
    w = wl.make_eam_tabulated(6, n_table=1501)
    s = md.from_workload(w, precision=md.MD_FP64)
    s.md_run(30, w.dt)
    x, v = np.zeros((w.natoms, 3)), np.zeros((w.natoms, 3))
    s.md_get_positions(x); s.md_get_velocities(v)
    ref = oracle.run_nve(w.x, w.v, w.box, np.full(w.natoms, w.mass[0]), w.style, wl.oracle_params(w), w.rc, w.skin, w.dt, 30,
                         ftm2v=w.ftm2v, mvv2e=w.mvv2e)
    assert np.abs(_minimg(x - ref["x"], w.box)).max() < 1e-10 and np.abs(v - ref["v"]).max() < 1e-9 * np.abs(ref["v"]).max()
    s.close()
    # a coarse table is a different potential: the GPU must follow the TABLE, not the analytic form it was sampled from
    wc = wl.make_eam_tabulated(6, n_table=61)
    xc = wl.perturbed(wc, 0.2)
    ft = oracle.forces_brute(xc, wc.box, wc.style, wl.oracle_params(wc), wc.rc)[0]
    fa = oracle.forces_brute(xc, wc.box, oracle.PAIR_EAM, wl.EAM_PARAMS, wc.rc)[0]
    s = md.from_workload(wc, precision=md.MD_FP64, x=xc)
    f = np.zeros((wc.natoms, 3))
    s.md_compute_forces(f)
    assert _fp64_force_err(f, ft) < 1e-11 and _fp64_force_err(f, fa) > 1e-6
    s.close()
    # tables that end before the cutoff, or are missing, are refused
    s = md.System(w.box, w.natoms, w.types, w.mass)
    s.md_set_pair(md.MD_PAIR_EAM_TAB, (0.004, 0.05), w.rc, w.skin)
    s.md_set_positions(w.x)
    with pytest.raises(md.MDError) as e:
        s.md_compute_forces()
    assert e.value.code == md.MD_ERR_NOT_READY
    s.md_set_eam_tables(np.ones(100), np.ones(100), np.ones(100))          # reaches r = 0.396 only
    with pytest.raises(md.MDError) as e:
        s.md_compute_forces()
    assert e.value.code == md.MD_ERR_BAD_ARGUMENT
    s.close()


@pytest.mark.parametrize("kernel,shape", [(1, 0x111), (5, 0x112), (6, 0x122), (3, 0x111)])
def test_persistent_kernel_on_a_small_box_many_tiles_per_block(kernel, shape):
    """The persistent force kernel normally needs a box of a few hundred tiles; persistent_min_tiles_per_sm = 0 runs it on
    any box.  16,384 atoms in one-cell (or two-, four-cell) tiles give every block several tiles, so that the tile
    buffers are reused, tasks of three tiles are in flight at once and consumer warps help with the post-processing."""
    w = wl.make(2, n_override=16)
    x = wl.perturbed(w, 0.12)
    s = md.from_workload(w, x=x, kernel=kernel, options={"persistent_min_tiles_per_sm": 0, "tile_shape": shape})
    f = np.zeros((w.natoms, 3))
    s.md_compute_forces(f)                                           # no energy: the persistent kernel
    assert _rel_rms(f, oracle.forces(x, w.box, w.style, w.params, w.rc)[0]) < 1e-5
    st = s.md_get_stats()
    assert st["ntiles"] > 3 * 148 or shape != 0x111
    f2 = np.zeros_like(f)
    s.md_compute_forces(f2)
    assert np.array_equal(f, f2)                                     # tasks are dealt dynamically, the arithmetic is not
    s.md_run(25, w.dt)
    xg = np.zeros((w.natoms, 3)); s.md_get_positions(xg); s.md_get_forces(f)
    assert _rel_rms(f, oracle.forces(xg, w.box, w.style, w.params, w.rc)[0]) < 1e-5
    s.close()


def test_tabulated_eam_tables_staged_in_shared_memory():
    """MD_PAIR_EAM_TAB in the persistent kernel copies its coefficient tables behind the tile buffers (option tab_smem);
    the lookups must return what the read-only path returns: bitwise the same forces, both within tolerance of the oracle."""
    w = wl.make_eam_tabulated(8, n_table=2001)
    x = wl.perturbed(w, 0.2)
    fo = oracle.forces(x, w.box, w.style, wl.oracle_params(w), w.rc)[0]
    out = {}
    for tab_smem in (1, 0):
        s = md.from_workload(w, precision=md.MD_MIXED, x=x, options={"persistent_min_tiles_per_sm": 0, "tab_smem": tab_smem})
        f = np.zeros((w.natoms, 3))
        s.md_compute_forces(f)
        assert _rel_rms(f, fo) < 1e-5
        s.md_run(10, w.dt)
        s.md_get_forces(f)
        out[tab_smem] = f
        s.close()
    assert np.array_equal(out[0], out[1])


# ---- NVT, one Nose-Hoover thermostat (reading s25) -----------------------------------

@pytest.mark.parametrize("cfg,n,nsteps,kT_factor,tau,list_kind", [(1, 7, 60, 0.5, 0.1, 0), (1, 7, 40, 0.5, 0.1, 1), (4, 6, 40, 2.0, 0.02, 0)])
def test_nvt_run_matches_oracle_trajectory(cfg, n, nsteps, kT_factor, tau, list_kind):
    w = wl.make(cfg, n_override=n)
    kT = kT_factor * w.kT
    s = md.from_workload(w, precision=md.MD_FP64, kernel=md.MD_KERNEL_TPA, list_kind=list_kind)
    s.md_set_thermostat(md.MD_THERMO_NOSE_HOOVER, kT, tau)
    half = nsteps // 2
    s.md_run(half, w.dt)                       # in two pieces: the thermostat state persists across calls
    s.md_run(nsteps - half, w.dt)
    x, v = np.zeros((w.natoms, 3)), np.zeros((w.natoms, 3))
    s.md_get_positions(x); s.md_get_velocities(v)
    ref = oracle.run_nvt(w.x, w.v, w.box, np.full(w.natoms, w.mass[0]), w.style, w.params, w.rc, w.skin, w.dt, nsteps,
                         kT=kT, tau=tau, ftm2v=w.ftm2v, mvv2e=w.mvv2e)
    assert np.abs(_minimg(x - ref["x"], w.box)).max() < 1e-9
    assert np.abs(v - ref["v"]).max() < 1e-8 * np.abs(ref["v"]).max()
    th = s.md_get_thermostat()
    assert th["xi"] == pytest.approx(ref["thermo"][0], rel=1e-8) and th["eta"] == pytest.approx(ref["thermo"][1], rel=1e-8)
    assert abs(ref["thermo"][0]) * tau > 1e-3             # the thermostat acted
    ke = s.md_kinetic_energy()
    assert ke == pytest.approx(ref["ke"][-1], rel=1e-9)
    # conserved quantity through the API: KE + PE + thermostat share equals the oracle's H
    E, _ = s.md_compute_forces(energy=True)
    assert ke + E + th["energy"] == pytest.approx(ref["h"][-1], rel=1e-9)
    assert abs(s.md_get_stats()["nbuilds"] - ref["nbuild"]) <= 2
    s.md_set_thermostat(md.MD_THERMO_NONE)
    s.close()


def test_nvt_mixed_precision_thermalises_and_rejects_bad_arguments():
    w = wl.make(2, n_override=8)
    s = md.from_workload(w, kernel=md.MD_KERNEL_AUTO)
    for kT, tau in [(-1.0, 0.1), (1.0, 0.0), (float("nan"), 0.1)]:
        with pytest.raises(md.MDError) as e:
            s.md_set_thermostat(md.MD_THERMO_NOSE_HOOVER, kT, tau)
        assert e.value.code == md.MD_ERR_BAD_ARGUMENT
    s.md_set_thermostat(md.MD_THERMO_NOSE_HOOVER, 0.8, 0.2)
    s.md_run(600, w.dt)
    g = 3 * w.natoms - 3
    T = [2.0 * s.md_kinetic_energy() / g]
    for _ in range(10):
        s.md_run(40, w.dt)
        T.append(2.0 * s.md_kinetic_energy() / g)
    assert np.mean(T) == pytest.approx(0.8, rel=0.06)
    s.close()


@pytest.mark.parametrize("build_graph", [1, 0])
def test_capacity_overflow_inside_a_run_replans_and_matches_oracle(build_graph):
    """md_run does not wait for its rebuilds: the step kernels that follow one on the stream judge its flags themselves
    (a tile or row that outgrew its capacity stops the batch before its first step) and the host plans anew after the
    batch.  A converging flow (v_x = -c sin(2 pi x / L) on a dilute lattice) piles the atoms up around x = L/2 until the
    rows outgrow the capacity planned for the uniform start; the trajectory must still be the oracle's.  With and
    without the CUDA-graph replay of the build sequence."""
    n, a, c, dt, nsteps = 16, 1.5, 2.0, 0.004, 450
    L = n * a
    g = (np.arange(n) + 0.5) * a
    x = np.stack(np.meshgrid(g, g, g, indexing="ij"), -1).reshape(-1, 3).copy()
    x += np.random.default_rng(3).uniform(-0.05, 0.05, x.shape)
    v = np.zeros_like(x)
    v[:, 0] = -c * np.sin(2 * np.pi * x[:, 0] / L)
    box = np.array([L, L, L])
    N = len(x)
    s = md.System(box, N, np.zeros(N, np.int32), np.array([1.0]))
    s.md_set_precision(md.MD_FP64)
    s.md_set_pair(md.MD_PAIR_LJ126, (1.0, 1.0), 2.5, 0.3)
    s.md_set_neighbor(md.MD_LIST_FULL, md.MD_KERNEL_TPA)
    s.md_set_option("build_graph", build_graph)
    s.md_set_positions(x); s.md_set_velocities(v)
    s.md_build_neighbors()
    st0 = s.md_get_stats()
    s.md_run(nsteps, dt)
    st1 = s.md_get_stats()
    assert st1["row_capacity"] > st0["row_capacity"] and st1["max_row"] > st0["row_capacity"]      # the plan was outgrown in the run
    ref = oracle.run_nve(x, v, box, np.ones(N), oracle.PAIR_LJ, (1.0, 1.0), 2.5, 0.3, dt, nsteps)
    xg, vg, fg = (np.zeros((N, 3)) for _ in range(3))
    s.md_get_positions(xg); s.md_get_velocities(vg); s.md_get_forces(fg)
    assert np.abs(_minimg(xg - ref["x"], box)).max() < 1e-9 and np.abs(vg - ref["v"]).max() < 1e-8
    assert st1["nsteps_total"] == nsteps
    assert ref["nbuild"] <= st1["nbuilds"] - st0["nbuilds"] <= ref["nbuild"] + 8             # the overflowed builds are done twice
    fo = oracle.forces(xg, box, oracle.PAIR_LJ, (1.0, 1.0), 2.5)[0]
    assert _fp64_force_err(fg, fo) < 1e-12
    s.close()


# ---- errors and degenerate inputs ------------------------------------------------------------------------------

def test_error_paths():
    box = np.array([8.0, 8.0, 8.0])
    s = md.System(box, 4, np.zeros(4, np.int32), np.array([1.0]))
    with pytest.raises(md.MDError) as e:
        s.md_set_pair(md.MD_PAIR_LJ126, (1.0, 1.0), 2.5, 0.3)        # 8 < 3 * 2.8
    assert e.value.code == md.MD_ERR_BOX_TOO_SMALL
    with pytest.raises(md.MDError) as e:
        s.md_set_pair(md.MD_PAIR_LJ126, (1.0, 1.0, 1.0), 2.0, 0.3)
    assert e.value.code == md.MD_ERR_BAD_ARGUMENT
    with pytest.raises(md.MDError) as e:
        s.md_set_pair(99, (1.0, 1.0), 2.0, 0.3)
    assert e.value.code == md.MD_ERR_BAD_ARGUMENT
    s.md_set_pair(md.MD_PAIR_LJ126, (1.0, 1.0), 2.0, 0.3)
    with pytest.raises(md.MDError) as e:
        s.md_build_neighbors()                                         # positions not set
    assert e.value.code == md.MD_ERR_NOT_READY
    with pytest.raises(md.MDError) as e:
        s.md_set_neighbor(md.MD_LIST_HALF, md.MD_KERNEL_WARP)
    assert e.value.code == md.MD_ERR_BAD_ARGUMENT
    x = np.array([[1.0, 1, 1], [2.2, 1, 1], [np.nan, 1, 1], [5.0, 5, 5]])
    s.md_set_positions(x)
    with pytest.raises(md.MDError) as e:
        s.md_build_neighbors()
    assert e.value.code == md.MD_ERR_NONFINITE
    with pytest.raises(md.MDError):
        md.System(np.array([1.0, -1.0, 1.0]), 4, np.zeros(4, np.int32), np.array([1.0]))
    with pytest.raises(md.MDError):
        md.System(box, 0, np.zeros(0, np.int32), np.array([1.0]))
    for name, value in [("no_such_option", 1), ("tile_shape", 0x135), ("tile_shape", 0x511), ("persistent_groups", 3), ("force_threads", -32)]:
        with pytest.raises(md.MDError) as e:
            s.md_set_option(name, value)
        assert e.value.code == md.MD_ERR_BAD_ARGUMENT


@pytest.mark.parametrize("options", [{"tile_shape": 0x111}, {"tile_shape": 0x112, "no_persistent": 1}, {"persistent_groups": 1},
                                     {"force_threads": 64, "balance_after": 0}])
def test_tuning_options_change_the_plan_not_the_result(options):
    """md_set_option knobs (tile shape, block size, persistent-kernel layout, row balancing) must leave forces and energy
    within the mixed-precision tolerance of the brute-force oracle."""
    w = wl.make(2, n_override=8)
    x = wl.perturbed(w, 0.12)
    fo, Eo = oracle.forces_brute(x, w.box, w.style, w.params, w.rc)[:2]
    s = md.from_workload(w, x=x, options=options)
    f = np.zeros((w.natoms, 3))
    E, _ = s.md_compute_forces(f, energy=True)
    assert _rel_rms(f, fo) < 1e-5 and abs(E - Eo) < 1e-6 * abs(Eo)
    if "tile_shape" in options:
        b = options["tile_shape"]
        assert s.md_get_stats()["brick"] == [b & 15, (b >> 4) & 15, (b >> 8) & 15]
    s.md_run(30, w.dt)
    xg = np.zeros((w.natoms, 3)); s.md_get_positions(xg); s.md_get_forces(f)
    assert _rel_rms(f, oracle.forces(xg, w.box, w.style, w.params, w.rc)[0]) < 1e-5
    s.close()


def test_sparse_gas_empty_cells_and_zero_steps():
    """Mostly empty cells, atoms outside the box on input, nsteps = 0, isolated EAM atom (rho = 0)."""
    box = np.array([40.0, 30.0, 20.0])
    rng_ids = np.arange(50, dtype=np.uint64)
    x = np.stack([wl.uniform01(3, rng_ids, c) for c in range(3)], axis=1) * box
    x[::5] += box * np.array([2.0, -1.0, 3.0])                        # other periodic images
    for style, params, rc, skin in [(md.MD_PAIR_LJ126, (1.0, 1.0), 2.5, 0.3), (md.MD_PAIR_EAM_FS, wl.EAM_PARAMS, 4.95, 1.0)]:
        for prec in (md.MD_FP64, md.MD_MIXED):
            s = md.System(box, 50, np.zeros(50, np.int32), np.array([1.0]))
            s.md_set_precision(prec)
            s.md_set_pair(style, params, rc, skin)
            s.md_set_positions(x)
            s.md_set_velocities(np.zeros((50, 3)))
            s.md_run(0, 0.001)
            f = np.zeros((50, 3))
            E, _ = s.md_compute_forces(f, energy=True)
            fo, Eo = oracle.forces_brute(x, box, style, params, rc)[:2]
            assert np.all(np.isfinite(f))
            scale = max(np.abs(fo).max(), 1e-300)
            assert np.abs(f - fo).max() <= (1e-12 if prec == md.MD_FP64 else 1e-5) * scale
            assert abs(E - Eo) <= (1e-12 if prec == md.MD_FP64 else 2e-6) * max(abs(Eo), 1e-300)


@pytest.mark.parametrize("precision", [0, 1])
@pytest.mark.parametrize("kernel,list_kind", [(0, 0), (1, 0), (5, 0), (2, 0), (3, 0), (4, 0), (1, 1)])
def test_non_cubic_box_ragged_tiles(kernel, list_kind, precision):
    """A box with 5 x 4 x 3 cells: tile shapes are clipped to the box, the last tile of a dimension is narrower
    than the others, every tile sees periodic images.  Pair set, forces, energy and virial against brute force."""
    a = wl.LJ_A
    nx, ny, nz = 9, 7, 6
    base = np.array([[0, 0, 0], [.5, .5, 0], [.5, 0, .5], [0, .5, .5]])
    g = np.stack(np.meshgrid(np.arange(nx), np.arange(ny), np.arange(nz), indexing="ij"), axis=-1).reshape(-1, 1, 3)
    x = ((g + base[None]) * a).reshape(-1, 3)
    box = np.array([nx, ny, nz]) * a
    N = x.shape[0]
    x = x + wl.uniform_displacements(5, np.arange(N, dtype=np.uint64), 0.15)
    x -= np.floor(x / box) * box
    rc, skin = 2.5, 0.3
    s = md.System(box, N, np.zeros(N, np.int32), np.array([1.0]))
    s.md_set_precision(precision)
    s.md_set_neighbor(list_kind, kernel)
    s.md_set_pair(md.MD_PAIR_LJ126, (1.0, 1.0), rc, skin)
    s.md_set_positions(x)
    s.md_build_neighbors()
    st = s.md_get_stats()
    assert st["ncells"] == [5, 4, 3]
    nn, nb = _gpu_rows(s, N, 160)
    got = {(min(i, int(j)), max(i, int(j))) for i in range(N) for j in nb[i, :nn[i]]}
    sure, fuzzy = _oracle_pairs(x, box, rc + skin)
    assert sure <= got and got <= (sure | fuzzy)
    assert int(nn.sum()) == (len(got) if list_kind else 2 * len(got))
    f = np.zeros((N, 3))
    E, W = s.md_compute_forces(f, energy=True, virial=True)
    fo, Eo, Wo, _, _ = oracle.forces_brute(x, box, oracle.PAIR_LJ, (1.0, 1.0), rc)
    if precision == md.MD_FP64:
        assert _fp64_force_err(f, fo) < 1e-12 and abs(E - Eo) < 1e-12 * abs(Eo)
        assert np.abs(W - Wo).max() < 1e-11 * np.abs(Wo).max()
    else:
        assert _rel_rms(f, fo) < 1e-5 and abs(E - Eo) < 1e-6 * abs(Eo)
    s.md_set_velocities(np.zeros((N, 3)))
    s.md_run(30, 0.004)                       # crosses rebuilds as the perturbed lattice relaxes
    xg = np.zeros((N, 3)); s.md_get_positions(xg); s.md_get_forces(f)
    fo = oracle.forces(xg, box, oracle.PAIR_LJ, (1.0, 1.0), rc)[0]
    assert (_fp64_force_err(f, fo) < 1e-12) if precision == md.MD_FP64 else (_rel_rms(f, fo) < 1e-5)
    s.close()


@pytest.mark.parametrize("seed", list(range(16)))
def test_randomised_boxes_densities_cutoffs(seed):
    """Seeded random geometry: orthogonal boxes with unequal edges, densities from a dilute gas to a dense fluid
    (a jittered simple-cubic lattice with random vacancies, so no two atoms overlap), cutoffs and skins that move
    the cell grid from 3 to 6 cells per edge, every variant and both precisions in turn.  Pair set against the
    brute-force enumeration; forces, energy, virial against the O(N^2) definition."""
    rs = np.random.RandomState(1000 + seed)
    rc = float(rs.uniform(1.6, 2.6)); skin = float(rs.uniform(0.0, 0.5)); rl = rc + skin
    edges = rl * rs.uniform(3.02, 6.3, size=3)
    a = float(rs.uniform(0.95, 1.6))                                    # lattice spacing: density a^-3 x occupancy
    n = np.maximum(np.floor(edges / a).astype(int), 1)
    box = n * a
    box = np.maximum(box, 3.001 * rl)
    g = np.stack(np.meshgrid(*[np.arange(k) for k in n], indexing="ij"), axis=-1).reshape(-1, 3).astype(float)
    keep = rs.uniform(size=len(g)) < rs.uniform(0.25, 1.0)
    x = (g[keep] + 0.5) * (box / n) + rs.uniform(-0.12, 0.12, size=(int(keep.sum()), 3)) * a
    x += box * rs.randint(-2, 3, size=x.shape)                          # any periodic image on input
    N = x.shape[0]
    kernel, list_kind = [(0, 0), (1, 0), (5, 0), (2, 0), (3, 0), (4, 0), (1, 1), (0, 0)][seed % 8]
    precision = (seed // 8) % 2
    s = md.System(box, N, np.zeros(N, np.int32), np.array([1.0]))
    s.md_set_precision(precision)
    s.md_set_neighbor(list_kind, kernel)
    s.md_set_pair(md.MD_PAIR_LJ126, (1.0, 1.0), rc, skin)
    s.md_set_positions(x)
    s.md_build_neighbors()
    nn, nb = _gpu_rows(s, N, 256)
    got = {(min(i, int(j)), max(i, int(j))) for i in range(N) for j in nb[i, :nn[i]]}
    xw = x - np.floor(x / box) * box
    sure, fuzzy = _oracle_pairs(xw, box, rl)
    assert sure <= got and got <= (sure | fuzzy)
    assert int(nn.sum()) == (len(got) if list_kind else 2 * len(got))
    f = np.zeros((N, 3))
    E, W = s.md_compute_forces(f, energy=True, virial=True)
    fo, Eo, Wo, _, _ = oracle.forces_brute(xw, box, oracle.PAIR_LJ, (1.0, 1.0), rc)
    if precision == md.MD_FP64:
        assert _fp64_force_err(f, fo) < 1e-12
        assert abs(E - Eo) < 1e-12 * max(abs(Eo), 1.0) and np.abs(W - Wo).max() < 1e-11 * max(np.abs(Wo).max(), 1.0)
    else:
        # a random dense configuration has large repulsive and attractive terms that cancel in E; the fp32 pair terms
        # are accurate to 1e-6 of the terms themselves, so the energy is judged against sum |u_pair|
        _, _, r2 = oracle.pairs_brute(xw, box, rc, with_r2=True)
        uabs = float(np.abs(4.0 * (r2 ** -6 - r2 ** -3)).sum())
        assert _rel_rms(f, fo) < 1e-5 and abs(E - Eo) < 1e-6 * max(uabs, 1.0)
    s.close()


def test_two_types_select_masses():
    w = wl.make(1, n_override=6)
    types = (np.arange(w.natoms) % 2).astype(np.int32)
    mass = np.array([1.0, 3.0])
    s = md.System(w.box, w.natoms, types, mass)
    s.md_set_pair(w.style, w.params, w.rc, w.skin)
    s.md_set_positions(w.x); s.md_set_velocities(w.v)
    s.md_run(30, w.dt)
    x = np.zeros((w.natoms, 3))
    s.md_get_positions(x)
    ref = oracle.run_nve(w.x, w.v, w.box, mass[types], w.style, w.params, w.rc, w.skin, w.dt, 30)
    assert np.abs(_minimg(x - ref["x"], w.box)).max() < 1e-10


def test_device_buffers_torch():
    import torch
    w = wl.make(1, n_override=6)
    x = wl.perturbed(w, 0.1)
    s = md.System(w.box, w.natoms, torch.zeros(w.natoms, dtype=torch.int32, device="cuda"), w.mass)
    s.md_set_pair(w.style, w.params, w.rc, w.skin)
    s.md_set_positions(torch.from_numpy(x).cuda())
    f = torch.zeros((w.natoms, 3), dtype=torch.float64, device="cuda")
    s.md_compute_forces(f)
    torch.cuda.synchronize()
    fo = oracle.forces_brute(x, w.box, w.style, w.params, w.rc)[0]
    assert _fp64_force_err(f.cpu().numpy(), fo) < 1e-12


def test_autotune_picks_a_variant_and_stays_correct():
    w, x, s = _system(1, 8, 0.12, md.MD_MIXED, md.MD_KERNEL_AUTO)
    ms = s.md_autotune(2)
    assert all(v > 0 for v in ms.values())
    st = s.md_get_stats()
    assert st["kernel_variant"] in (1, 2, 3, 5, 6)
    f = np.zeros((w.natoms, 3))
    s.md_compute_forces(f)
    assert _rel_rms(f, oracle.forces_brute(x, w.box, w.style, w.params, w.rc)[0]) < 1e-5
