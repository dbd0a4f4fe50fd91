"""CPU-side checks: the C-ABI library loads and exports every symbol include/md_b200.h declares (no
compute calls without a GPU); the world_size-2 replica bookkeeping of bench.py over gloo."""
import ctypes
import os
import re
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "md_b200.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(md_[a-z_0-9]+)\s*\(", text)))


def test_library_builds_loads_and_exports_every_declared_symbol():
    from paper_1009_4330_b200 import build
    lib_path = build.build()
    lib = ctypes.CDLL(lib_path)
    names = _declared_symbols()
    assert {"md_create", "md_set_pair", "md_build_neighbors", "md_compute_forces", "md_run"} <= set(names)
    for name in names:
        assert hasattr(lib, name), "libmd_b200.so does not export %s" % name
    from paper_1009_4330_b200 import md
    assert sorted(md.EXPORTS) == names, "the Python binding and the header disagree"


def test_stats_struct_matches_header_layout():
    """md_stats is filled by C and read by ctypes: field order and count must agree with the header."""
    from paper_1009_4330_b200 import md
    text = open(os.path.join(ROOT, "include", "md_b200.h")).read()
    body = re.search(r"typedef struct md_stats \{(.*?)\} md_stats;", text, flags=re.S).group(1)
    body = re.sub(r"/\*.*?\*/", "", body, flags=re.S)
    fields = [re.sub(r"\[.*\]", "", f.split()[-1]) for f in body.split(";") if f.strip()]
    assert fields == [n for n, _ in md.md_stats._fields_]


def test_argument_errors_without_a_gpu():
    """Argument validation happens before any CUDA call, so it can be exercised on a CPU box."""
    from paper_1009_4330_b200 import md
    h = ctypes.c_void_p()
    box = (ctypes.c_double * 3)(1.0, 1.0, -1.0)
    mass = (ctypes.c_double * 1)(1.0)
    types = (ctypes.c_int32 * 4)(0, 0, 0, 0)
    rc = md.lib.md_create(ctypes.byref(h), box, 4, ctypes.cast(types, ctypes.c_void_p), 1, mass, None)
    assert rc == md.MD_ERR_BAD_ARGUMENT and not h.value
    assert b"box" in md.lib.md_last_error(None)
    assert md.lib.md_run(None, 1, 0.1) == md.MD_ERR_BAD_ARGUMENT
    assert md.lib.md_set_units(None, 1.0, 1.0) == md.MD_ERR_BAD_ARGUMENT


def test_noalloc_entry_point_checks_its_arguments_before_any_cuda_call():
    """md_kinetic_energy_noalloc rejects NULL pointers and sizes outside (0, MD_NOALLOC_MAX_ATOMS] with a clear message,
    and the limit in the binding is the header's."""
    from paper_1009_4330_b200 import md
    text = open(os.path.join(ROOT, "include", "md_b200.h")).read()
    assert int(re.search(r"#define MD_NOALLOC_MAX_ATOMS (\d+)LL", text).group(1)) == md.MD_NOALLOC_MAX_ATOMS
    assert int(re.search(r"#define MD_NOALLOC_SCRATCH_BYTES (\d+)", text).group(1)) == md.MD_NOALLOC_SCRATCH_BYTES
    assert md.MD_NOALLOC_MAX_ATOMS == (md.MD_NOALLOC_SCRATCH_BYTES - 256) // 8 * 256
    fake = 4096     # never dereferenced: the checks come first
    f = md.lib.md_kinetic_energy_noalloc
    assert f(None, fake, fake, 10, 1.0, fake, None) == md.MD_ERR_BAD_ARGUMENT and b"NULL" in md.lib.md_last_error(None)
    assert f(fake, fake, fake, 10, 1.0, None, None) == md.MD_ERR_BAD_ARGUMENT
    assert f(fake, fake, fake, 0, 1.0, fake, None) == md.MD_ERR_BAD_ARGUMENT and b"positive" in md.lib.md_last_error(None)
    assert f(fake, fake, fake, md.MD_NOALLOC_MAX_ATOMS + 1, 1.0, fake, None) == md.MD_ERR_BAD_ARGUMENT
    msg = md.lib.md_last_error(None).decode()
    assert "MD_NOALLOC_MAX_ATOMS" in msg and str(md.MD_NOALLOC_MAX_ATOMS + 1) in msg


def test_roofline_traffic_is_read_from_the_committed_ncu_summaries():
    """bench.py takes roofline.traffic from the `dram_bytes_per_launch:` lines that ncu_summary wrote into profiles/."""
    from paper_1009_4330_b200 import ncu_summary
    prof = os.path.join(ROOT, "profiles")
    t5 = ncu_summary.traffic(os.path.join(prof, "r02_ncu_full_force_cfg5.md"))
    assert t5 is not None and 5e8 < t5 < 3e9                      # a 4 M-atom LJ force launch moves about a gigabyte
    one = ncu_summary.traffic(os.path.join(prof, "r02_ncu_full_force_cfg4.md"), sections=1)
    two = ncu_summary.traffic(os.path.join(prof, "r02_ncu_full_force_cfg4.md"), sections=2)
    assert one is not None and two is not None and two > one      # EAM: density pass + force pass
    assert ncu_summary.traffic(os.path.join(prof, "r02_ncu_full_force_cfg4.md"), sections=3) is None
    assert ncu_summary.traffic(os.path.join(prof, "no_such_file.md")) is None


def test_product_path_never_imports_the_oracle():
    for dirpath, _, files in os.walk(os.path.join(ROOT, "paper_1009_4330_b200")):
        for fn in files:
            if fn.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, fn)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", src, flags=re.M), fn
                assert "md_oracle" not in src and "liboracle" not in src, fn
    osrc = open(os.path.join(ROOT, "oracle", "__init__.py")).read() + open(os.path.join(ROOT, "oracle", "md_oracle.c")).read()
    assert "import paper_1009_4330_b200" not in osrc and "from paper_1009_4330_b200" not in osrc
    assert "md_kernels" not in osrc and "#include \"../" not in osrc


_WORKER = r"""
import os, sys
sys.path.insert(0, %r)
from paper_1009_4330_b200 import dist as mdist, workloads as wl
rk = mdist.init("gloo")
assert rk.world == 2 and rk.backend == "gloo"
mdist.barrier(rk)
w = wl.make(1, n_override=3, seed_offset=mdist.replica_seed_offset(rk))
units = float(w.natoms) * 10
secs = 1.0 + rk.rank          # rank 1 is slower: the aggregate must use the max
value, tmax = mdist.aggregate_throughput(rk, units, secs)
assert tmax == 2.0 and value == 2 * units / 2.0, (value, tmax)
vsum = mdist.all_sum(rk, float(abs(w.v).sum()))
print("RANK", rk.rank, "OK", "%%.12e" %% float(abs(w.v).sum()), "%%.12e" %% vsum, flush=True)
mdist.finalize(rk)
"""


def test_two_replica_bookkeeping_over_gloo(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(_WORKER % ROOT)
    env = dict(os.environ, MASTER_ADDR="127.0.0.1", MASTER_PORT="29617", WORLD_SIZE="2")
    procs = [subprocess.Popen([sys.executable, str(script)], env=dict(env, RANK=str(r), LOCAL_RANK=str(r)),
                              stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True) for r in range(2)]
    outs = [p.communicate(timeout=240)[0] for p in procs]
    assert all(p.returncode == 0 for p in procs), outs
    rows = [[l for l in o.splitlines() if l.startswith("RANK")][0].split() for o in outs]
    assert rows[0][3] != rows[1][3], "replicas must draw different velocities"
    assert rows[0][4] == rows[1][4], "all_sum must agree on both ranks"


def test_bench_reference_arm_other_ranks_do_no_work():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2"], env=env,
                         capture_output=True, text=True, timeout=120)
    assert out.returncode == 0 and out.stdout.strip() == ""


def test_sweep_module_fails_loudly_without_a_gpu():
    """The measurement helper has no CPU fallback either."""
    import subprocess
    import sys
    import torch
    if torch.cuda.is_available():
        pytest.skip("needs a box without a GPU")
    r = subprocess.run([sys.executable, "-m", "paper_1009_4330_b200.sweep", "--cells", "6", "--rc", "2.5"], capture_output=True, text=True,
                       cwd=os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
    assert r.returncode != 0 and "no CUDA device" in (r.stderr + r.stdout)
