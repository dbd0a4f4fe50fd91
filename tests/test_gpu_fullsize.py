"""Parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times (MD_KERNEL_AUTO, full
list, the config's own precision), on the same seeded inputs.

At these sizes the oracle cannot enumerate all pairs by brute force, so the comparison is
  * sampled atoms, one by one: orc_forces_sample / orc_neighbors_sample scan ALL N atoms per sampled atom
    (the plain definition, any N); the GPU's forces and list rows of those atoms are compared with them;
  * every atom: the oracle's O(N) list route (itself pinned to the brute force in test_oracle_pins.py)
    recomputes forces, energy and virial from the GPU's OWN fp64 positions after a piece of the run
    that crosses several list rebuilds (same-input snapshot, SURVEY.md §8(c) "GPU vs oracle").
Tolerances: north_star -- mixed: relative RMS force error <= 1e-5, energy <= 1e-6 relative; fp64: 1e-12;
pair sets identical outside the 1e-9 band around rc+skin.
"""
import numpy as np
import pytest

import oracle
from paper_1009_4330_b200 import workloads as wl

pytestmark = pytest.mark.gpu

NSAMPLE = 48


def _rel_rms(f, ref):
    return float(np.sqrt(((f - ref) ** 2).sum() / (ref ** 2).sum()))


def _sample_ids(N, seed):
    u = wl.uniform01(seed, np.arange(NSAMPLE, dtype=np.uint64), 9)
    return np.unique((u * N).astype(np.int64))


@pytest.mark.parametrize("cfg,steps", [(2, 40), (3, 12), (4, 30), (5, 14)])
def test_full_size_run_snapshot_matches_oracle(cfg, steps):
    import torch
    from paper_1009_4330_b200 import md
    w = wl.make(cfg)
    N = w.natoms
    s = md.from_workload(w, kernel=md.MD_KERNEL_AUTO)          # what bench.py launches
    s.md_run(steps, w.dt)
    st = s.md_get_stats()
    assert st["nsteps_total"] == steps
    if w.style == wl.PAIR_LJ:
        assert st["nbuilds_in_run"] >= 2                        # the piece crossed displacement-triggered rebuilds
    x = np.zeros((N, 3)); f_run = np.zeros((N, 3))
    s.md_get_positions(x); s.md_get_forces(f_run)
    f = np.zeros((N, 3))
    E, W = s.md_compute_forces(f, energy=True, virial=True)    # same positions, the list the run left behind
    fo, Eo, Wo, _, _ = oracle.forces(x, w.box, w.style, w.params, w.rc)
    assert np.isfinite(f).all()
    assert _rel_rms(f, fo) < 1e-5, _rel_rms(f, fo)
    assert _rel_rms(f_run, fo) < 1e-5
    assert abs(E - Eo) < 1e-6 * abs(Eo), (E, Eo)
    assert np.abs(W[:3] - Wo[:3]).max() < 1e-5 * np.abs(Wo[:3]).max()
    # sampled atoms by the plain definition (full scan over all N)
    ids = _sample_ids(N, w.seed)
    fs, _ = oracle.forces_sample(x, w.box, w.style, w.params, w.rc, ids)
    scale = np.sqrt((fo ** 2).sum(axis=1).mean())
    assert np.abs(f[ids] - fs).max() < 3e-5 * scale
    assert np.abs(fo[ids] - fs).max() < 1e-10 * scale          # the oracle's two routes agree
    # the list the run left behind is still valid: every pair inside rc at the CURRENT positions is in it
    stride = int(st["max_neighbors"]) + 8
    nn = torch.zeros(N, dtype=torch.int32, device="cuda")
    nb = torch.full((N, stride), -1, dtype=torch.int32, device="cuda")
    s.md_get_neighbors(nn, nb, stride)
    idt = torch.from_numpy(ids).cuda()
    nn_s, nb_s = nn[idt].cpu().numpy(), nb[idt].cpu().numpy()
    cnt, inside = oracle.neighbors_sample(x, w.box, w.rc - 1e-9, ids, stride=2048)
    for k in range(len(ids)):
        have = set(nb_s[k, :nn_s[k]].tolist())
        assert len(have) == nn_s[k]
        assert set(inside[k, :cnt[k]].tolist()) <= have
    del nn, nb
    s.close()


@pytest.mark.parametrize("cfg", [3, 5])
def test_full_size_list_rows_match_full_scan(cfg):
    """Pair-set parity at build time: sampled rows of the freshly built list against a full scan."""
    import torch
    from paper_1009_4330_b200 import md
    w = wl.make(cfg)
    N = w.natoms
    x = wl.perturbed(w, 0.1)
    s = md.from_workload(w, kernel=md.MD_KERNEL_AUTO, x=x)
    s.md_build_neighbors()
    st = s.md_get_stats()
    stride = int(st["max_neighbors"]) + 8
    nn = torch.zeros(N, dtype=torch.int32, device="cuda")
    nb = torch.full((N, stride), -1, dtype=torch.int32, device="cuda")
    s.md_get_neighbors(nn, nb, stride)
    total = int(nn.sum().item())
    assert abs(total / N - st["mean_neighbors"]) < 1e-9 * total / N + 1e-6
    ids = _sample_ids(N, w.seed + 1)
    idt = torch.from_numpy(ids).cuda()
    nn_s, nb_s = nn[idt].cpu().numpy(), nb[idt].cpu().numpy()
    rl, band = w.rc + w.skin, 1e-9
    c_in, sure = oracle.neighbors_sample(x, w.box, rl - band, ids, stride=2048)
    c_out, maybe = oracle.neighbors_sample(x, w.box, rl + band, ids, stride=2048)
    for k in range(len(ids)):
        have = set(nb_s[k, :nn_s[k]].tolist())
        assert len(have) == nn_s[k]
        assert set(sure[k, :c_in[k]].tolist()) <= have <= set(maybe[k, :c_out[k]].tolist())
    # a full list is symmetric: row lengths of the partners include the sampled atom
    k = 0
    partners = torch.from_numpy(nb_s[k, :nn_s[k]].astype(np.int64)).cuda()
    rows = nb[partners]
    assert bool((rows == int(ids[k])).any(dim=1).all().item())
    del nn, nb
    s.close()


@pytest.mark.parametrize("cfg,kernel,list_kind,steps", [
    (5, 4, 0, 8),      # direct cell-list kernel at 4,000,000 atoms
    (5, 1, 1, 8),      # half list, atomic scatter
    (5, 5, 0, 8),      # 4 lanes per atom
    (3, 3, 0, 8),      # warp per atom at rc = 5 sigma (the paper's BpA regime)
    (4, 2, 0, 12),     # EAM, 8 lanes per atom
])
def test_full_size_other_variants_match_oracle(cfg, kernel, list_kind, steps):
    """Every kernel variant at full size: a short run crossing a rebuild, then the oracle recomputes forces and
    energy from the GPU's own positions (same-input snapshot) and sampled atoms by full scans."""
    from paper_1009_4330_b200 import md
    w = wl.make(cfg)
    N = w.natoms
    s = md.from_workload(w, kernel=kernel, list_kind=list_kind)
    s.md_run(steps, w.dt)
    x = np.zeros((N, 3)); f_run = np.zeros((N, 3))
    s.md_get_positions(x); s.md_get_forces(f_run)
    f = np.zeros((N, 3))
    E, _ = s.md_compute_forces(f, energy=True)
    st = s.md_get_stats()
    assert st["kernel_variant"] == kernel and st["nsteps_total"] == steps
    fo, Eo, _, _, _ = oracle.forces(x, w.box, w.style, w.params, w.rc)
    assert _rel_rms(f, fo) < 1e-5 and _rel_rms(f_run, fo) < 1e-5
    assert abs(E - Eo) < 1e-6 * abs(Eo)
    ids = _sample_ids(N, w.seed + 2)[:16]
    fs, _ = oracle.forces_sample(x, w.box, w.style, w.params, w.rc, ids)
    scale = np.sqrt((fo ** 2).sum(axis=1).mean())
    assert np.abs(f[ids] - fs).max() < 3e-5 * scale
    s.close()


@pytest.mark.parametrize("cfg,steps", [(2, 1000), (4, 200)])
def test_full_size_nve_drift_matches_the_oracles_own(cfg, steps):
    """NVE energy drift at full size (north_star; reading s2 / s12): lj/cut and the analytic EAM are plainly
    truncated, so pairs crossing rc jump the energy and the drift is judged against the fp64 oracle's own drift
    on the same input, not against an absolute bound.  Total energy per atom at the end of the GPU run (its own
    E and kinetic energy) must agree with the oracle's trajectory to a small multiple of the oracle's own
    step-to-step energy fluctuation; momentum stays zero."""
    from paper_1009_4330_b200 import md
    w = wl.make(cfg)
    N = w.natoms
    s = md.from_workload(w, kernel=md.MD_KERNEL_AUTO)
    E0, _ = s.md_compute_forces(energy=True)
    K0 = s.md_get_stats()["kinetic_energy"]
    s.md_run(steps, w.dt)
    E1, _ = s.md_compute_forces(energy=True)
    K1 = s.md_get_stats()["kinetic_energy"]
    v = np.zeros((N, 3)); s.md_get_velocities(v)
    s.close()
    ref = oracle.run_nve(w.x, w.v, w.box, np.full(N, w.mass[0]), w.style, w.params, w.rc, w.skin, w.dt, steps,
                         ftm2v=w.ftm2v, mvv2e=w.mvv2e, trace=True)
    et = ref["pe"] + ref["ke"]
    assert abs((E0 + K0) - et[0]) < 1e-6 * abs(et[0])
    drift_gpu = ((E1 + K1) - (E0 + K0)) / N
    drift_ref = (et[-1] - et[0]) / N
    wiggle = np.abs(np.diff(et)).max() / N                 # the oracle's own largest one-step change of E_tot per atom
    kT = w.kT
    assert abs(drift_gpu - drift_ref) < max(20 * wiggle, 2e-4 * kT), (drift_gpu, drift_ref, wiggle)
    if w.style == wl.PAIR_LJ:      # u(rc) is small for LJ; the truncated EAM (rho(rc) = 0.118) drifts by itself (reading s12)
        assert abs(drift_gpu) < 0.02 * kT and abs(drift_ref) < 0.02 * kT
    # kinetic energy follows the same melting / equipartition curve; after hundreds of steps the two chaotic
    # trajectories have decorrelated, so only to the canonical fluctuation of K, sqrt(2 / 3N) relative
    assert K1 == pytest.approx(ref["ke"][-1], rel=5.0 * np.sqrt(2.0 / (3.0 * N)))
    assert np.abs((v * w.mass[0]).sum(axis=0)).max() < 1e-6 * N * np.sqrt(w.mass[0] * kT / w.mvv2e)
