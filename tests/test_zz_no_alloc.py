"""md_kinetic_energy_noalloc (include/md_b200.h): the kinetic-energy reduction for callers that cannot call cudaMalloc,
its scratch in a file-scope static __device__ array.  Checked against the existing path, md_kinetic_energy on a handle
(itself checked against the oracle's trajectories in test_gpu_parity.py), within the fp64 tolerance of those tests
(1e-12 relative), on two calls in a row: the second call meets the scratch as the first one left it.

Collected last on purpose (the file name sorts after every other test file): the run uses ``pytest -x``.
"""
import numpy as np
import pytest

from paper_1009_4330_b200 import workloads as wl

pytestmark = pytest.mark.gpu

REL = 1e-12


def _device_buffers(torch, v, types, mass):
    dev = torch.device("cuda:0")
    return (torch.from_numpy(np.ascontiguousarray(v)).to(dev), torch.from_numpy(np.ascontiguousarray(types, dtype=np.int32)).to(dev),
            torch.from_numpy(np.ascontiguousarray(mass, dtype=np.float64)).to(dev), torch.full((1,), np.nan, dtype=torch.float64, device=dev))


def test_noalloc_kinetic_energy_matches_the_handle_path_on_two_calls_in_a_row():
    import torch
    from paper_1009_4330_b200 import md

    # call 1: LJ melt (reduced units, one type), 13,500 atoms = 53 blocks with a ragged last one, after 20 time steps
    w1 = wl.make(1, n_override=15)
    s1 = md.from_workload(w1, precision=md.MD_FP64)
    s1.md_run(20, w1.dt)
    v1 = np.zeros((w1.natoms, 3))
    s1.md_get_velocities(v1)
    ref1 = s1.md_kinetic_energy()
    # call 2: the two-species ionic crystal (metal units, mvv2e != 1, two masses), a different N: fewer blocks than
    # call 1 left partials for
    w2 = wl.make(6, n_override=16)
    s2 = md.from_workload(w2, precision=md.MD_FP64)
    s2.md_run(10, w2.dt)
    v2 = np.zeros((w2.natoms, 3))
    s2.md_get_velocities(v2)
    ref2 = s2.md_kinetic_energy()
    assert w2.natoms < w1.natoms and len(w2.mass) == 2 and w2.mvv2e != 1.0

    b1 = _device_buffers(torch, v1, w1.types, w1.mass)
    b2 = _device_buffers(torch, v2, w2.types, w2.mass)
    md.md_kinetic_energy_noalloc(b1[0], b1[1], b1[2], w1.mvv2e, b1[3])          # the first call on a device resolves the symbol
    torch.cuda.synchronize()                                                      # address and loads the kernel
    assert float(b1[3].item()) == pytest.approx(ref1, rel=REL)
    b1[3].fill_(float("nan"))
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]
    md.md_kinetic_energy_noalloc(b1[0], b1[1], b1[2], w1.mvv2e, b1[3])
    md.md_kinetic_energy_noalloc(b2[0], b2[1], b2[2], w2.mvv2e, b2[3])          # same stream: ordered after the first
    md.md_kinetic_energy_noalloc(b1[0], b1[1], b1[2], w1.mvv2e, b1[3])          # and the first input again: bitwise the same
    torch.cuda.synchronize()
    ke1_again = float(b1[3].item())
    md.md_kinetic_energy_noalloc(b1[0], b1[1], b1[2], w1.mvv2e, b1[3])
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free_before                            # nothing was allocated on the device
    ke1, ke2 = float(b1[3].item()), float(b2[3].item())
    assert ref1 > 0 and ref2 > 0
    assert ke1 == pytest.approx(ref1, rel=REL)
    assert ke2 == pytest.approx(ref2, rel=REL)
    assert ke1 == ke1_again
    # and against the definition, from the same velocities on the host
    host1 = 0.5 * (np.asarray(w1.mass)[w1.types][:, None] * v1 ** 2).sum() * w1.mvv2e
    host2 = 0.5 * (np.asarray(w2.mass)[w2.types][:, None] * v2 ** 2).sum() * w2.mvv2e
    assert ke1 == pytest.approx(host1, rel=REL) and ke2 == pytest.approx(host2, rel=REL)


def test_noalloc_rejects_sizes_beyond_the_static_scratch():
    import torch
    from paper_1009_4330_b200 import md

    dev = torch.device("cuda:0")
    v = torch.zeros(3, dtype=torch.float64, device=dev)
    t = torch.zeros(1, dtype=torch.int32, device=dev)
    m = torch.ones(1, dtype=torch.float64, device=dev)
    out = torch.full((1,), -1.0, dtype=torch.float64, device=dev)
    stream = md.current_stream_ptr()
    import ctypes
    for n, word in ((md.MD_NOALLOC_MAX_ATOMS + 1, "MD_NOALLOC_MAX_ATOMS"), (1 << 40, "MD_NOALLOC_MAX_ATOMS"), (0, "positive"), (-5, "positive")):
        rc = md.lib.md_kinetic_energy_noalloc(v.data_ptr(), t.data_ptr(), m.data_ptr(), n, 1.0, out.data_ptr(), ctypes.c_void_p(stream))
        assert rc == md.MD_ERR_BAD_ARGUMENT
        text = md.lib.md_last_error(None).decode()
        assert "md_kinetic_energy_noalloc" in text and str(n) in text and word in text
    rc = md.lib.md_kinetic_energy_noalloc(None, t.data_ptr(), m.data_ptr(), 1, 1.0, out.data_ptr(), ctypes.c_void_p(stream))
    assert rc == md.MD_ERR_BAD_ARGUMENT
    torch.cuda.synchronize()
    assert float(out.item()) == -1.0                                              # nothing was enqueued
    # a plain call still works afterwards: one atom, m = 3, |v|^2 = 9, mvv2e = 2
    md.md_kinetic_energy_noalloc(torch.tensor([[1.0, 2.0, 2.0]], dtype=torch.float64, device=dev), t, 3.0 * m, 2.0, out)
    torch.cuda.synchronize()
    assert float(out.item()) == 0.5 * 3.0 * 9.0 * 2.0
