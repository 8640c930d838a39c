"""Host-side checks that need no GPU: the C-ABI library builds, loads and exports every symbol that
include/jenga.h declares; descriptor validation and launch-shape helpers answer without a device;
the bench's schedule / work model / sharding helpers (two gloo ranks) behave."""
import ctypes as C
import os
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def L():
    from paper_2606_28394_b200 import binding
    return binding.lib()


def test_library_exports_every_declared_symbol(L):
    sys.path.insert(0, ROOT)
    import __graft_entry__ as G
    names = G.declared_symbols()
    assert {"jenga_world_create", "jenga_broadphase", "jenga_narrowphase", "jenga_pgs_solve", "jenga_step",
            "jenga_world_destroy", "jenga_step_host", "jenga_set_f_ext"} <= set(names)
    for n in names:
        assert hasattr(L, n), f"libjenga.so does not export {n}"


def test_library_is_sm100a_only():
    from paper_2606_28394_b200 import build
    out = subprocess.run(["cuobjdump", "-lelf", build.LIB], capture_output=True, text=True).stdout
    assert "sm_100a" in out and "sm_90" not in out and "sm_80" not in out


def test_library_uses_tensor_memory_and_shared_window_loads():
    """SASS evidence that the kernels are Blackwell-native: tcgen05.ld/st compile to LDTM/STTM, and the shared-memory
    arrays are addressed with LDS/STS (not generic LD/ST)."""
    from paper_2606_28394_b200 import build
    sass = subprocess.run(["cuobjdump", "-sass", build.LIB], capture_output=True, text=True).stdout
    assert sass.count("LDTM") >= 10 and sass.count("STTM") >= 5
    assert sass.count("LDS") > 500 and " LD.E" not in sass


def test_descriptor_validation_and_launch_shape(L):
    from paper_2606_28394_b200 import binding, workloads as W
    wp = W.make_config(2, n_envs=2).params
    d = binding.make_desc(wp)
    assert L.jenga_block_threads(C.byref(d)) in (32, 128, 256, 384, 512)   # one warp per env; 4, 8, 12 or 16 envs per CTA in the TMEM tiers
    smem = L.jenga_smem_bytes(C.byref(d))
    assert 0 < smem <= 227 * 1024
    # auto tier by batch size: a batch that does not fill 148 SMs runs fewer envs per SM (header, solver_tier)
    # and a batch that still fills every SM with two envs per solver warp (>= 2 x 16 x 148 envs) gets groups of two, in the
    # tier whose blocks in flight fit the L2 (12 warps per SM)
    shape = {}
    for E in (2, 592, 593, 1184, 1185, 1776, 1777, 4735, 4736, 65536):
        de = binding.make_desc(wp); de.n_envs = E
        shape[E] = (L.jenga_block_threads(C.byref(de)), L.jenga_env_group(C.byref(de)))
    assert shape == {2: (32, 1), 592: (32, 1), 593: (256, 1), 1184: (256, 1), 1185: (384, 1), 1776: (384, 1), 1777: (512, 1),
                     4735: (512, 1), 4736: (384, 2), 65536: (384, 2)}
    forced = binding.make_desc(wp, group=2); forced.n_envs = 9
    assert L.jenga_env_group(C.byref(forced)) == 2 and L.jenga_scratch_bytes(C.byref(forced)) > L.jenga_scratch_bytes(C.byref(binding.make_desc(wp)))
    bad = binding.make_desc(wp); bad.env_group = 3
    assert L.jenga_env_group(C.byref(bad)) == 0 and L.jenga_scratch_bytes(C.byref(bad)) == 0
    bad = binding.make_desc(wp); bad.body_stride = wp.n_bodies + 1          # not a multiple of 4
    assert L.jenga_smem_bytes(C.byref(bad)) == 0 and L.jenga_block_threads(C.byref(bad)) == 0
    bad = binding.make_desc(wp); bad.struct_size = 4
    assert L.jenga_smem_bytes(C.byref(bad)) == 0
    # NULL buffers are rejected before any CUDA call
    h = C.c_void_p()
    assert L.jenga_world_create(C.byref(d), C.byref(binding.Buffers()), C.byref(h)) == -1 and not h
    assert L.jenga_world_create(None, None, C.byref(h)) == -1
    assert L.jenga_step(None, 1, None) == -1 and L.jenga_world_destroy(None) == -1
    assert b"bad argument" in L.jenga_strerror(-1) and L.jenga_strerror(0) == b"ok"


def test_stage_buffers_are_optional_for_a_world_that_only_steps(L):
    """pairs / n_pairs / contacts / n_contacts / lambda: all five or none, and none only with materialise = 0.  The checks
    run before the first CUDA call, so without a device a descriptor that passes them fails later (not with -1); with a
    device it gives a handle (no kernel is launched by create / destroy)."""
    from paper_2606_28394_b200 import binding, workloads as W
    wp = W.make_config(2, n_envs=2).params

    def create(materialise, stage, **override):
        d = binding.make_desc(wp, materialise=materialise)
        b = binding.Buffers()
        names = ["state", "props", "mu", "cache_key", "cache_lam", "cache_pt", "n_cache", "status", "scratch"]
        names += stage
        for k, n in enumerate(names):
            setattr(b, n, 4096 * (k + 1))                      # aligned, never dereferenced on the host
        for n, v in override.items():
            setattr(b, n, v)
        b.scratch_bytes = L.jenga_scratch_bytes(C.byref(d))
        h = C.c_void_p()
        rc = L.jenga_world_create(C.byref(d), C.byref(b), C.byref(h))
        if rc == 0:
            L.jenga_world_destroy(h)
        return rc

    all_five = ["pairs", "n_pairs", "contacts", "n_contacts", "lambda_"]
    assert create(False, all_five) != -1 and create(True, all_five) != -1 and create(False, []) != -1
    assert create(True, []) == -1                              # materialise writes them
    assert create(False, ["pairs", "n_pairs"]) == -1           # some but not all
    assert create(False, all_five, contacts=4096 + 4) == -1    # misaligned
    assert create(False, [], state=None) == -1


def test_python_struct_matches_c_layout():
    """sizeof / field order of the ctypes mirror vs the header, via a tiny C program."""
    from paper_2606_28394_b200 import binding
    src = r'''
#include <stdio.h>
#include <stddef.h>
#include "jenga.h"
int main(void){ printf("%zu %zu %zu %zu %zu %zu\n", sizeof(jenga_world_desc), offsetof(jenga_world_desc, gravity),
  offsetof(jenga_world_desc, match_tol), offsetof(jenga_world_desc, device), sizeof(jenga_buffers), offsetof(jenga_buffers, counters)); return 0; }
'''
    import tempfile
    with tempfile.TemporaryDirectory() as td:
        open(os.path.join(td, "t.c"), "w").write(src)
        subprocess.check_call(["gcc", "-I", os.path.join(ROOT, "include"), "-o", os.path.join(td, "t"), os.path.join(td, "t.c")])
        got = [int(x) for x in subprocess.check_output([os.path.join(td, "t")]).split()]
    D, Bf = binding.WorldDesc, binding.Buffers
    assert got == [C.sizeof(D), D.gravity.offset, D.match_tol.offset, D.device.offset, C.sizeof(Bf), Bf.counters.offset]


def test_no_cpu_fallback_without_gpu():
    import torch
    from paper_2606_28394_b200 import binding, workloads as W
    if torch.cuda.is_available():
        pytest.skip("this check is for the GPU-less box")
    wl = W.make_config(1)
    with pytest.raises(binding.JengaError):
        binding.World(wl.params, wl.state, wl.props, wl.mu)


def test_bench_schedule_and_work_model():
    sys.path.insert(0, ROOT)
    import bench
    from paper_2606_28394_b200 import workloads as W
    wl = W.make_config(5, n_envs=2)
    sch = list(bench.schedule(wl, 480, 12))
    assert sum(n for _, n, _ in sch) == 480 and sch[0][0] == 0
    assert all(a == (60 <= s < 84) for s, n, a in sch) and all(not (s < 60 < s + n or s < 84 < s + n) for s, n, a in sch)
    # standing 54-block tower: 612 body contacts + 12 ground contacts, 156 colliding pairs
    cnt = dict(env_steps=1, body_steps=54, candidates=190, colliding=156, contacts=624, contact_iters=624 * 20, ground_contacts=12)
    wm = bench.work_model(cnt, 54, 20)
    assert wm["pgs_rows"] == 20 * (612 * 87 + 12 * 51)
    assert abs(wm["total"] - 1.36e6) / 1.36e6 < 0.02       # the survey's 1.36 M thread-instr per env-step


_WORKER = r'''
import os, sys
import numpy as np, torch, torch.distributed as dist
sys.path.insert(0, sys.argv[1])
from paper_2606_28394_b200 import shard, workloads as W
dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{sys.argv[2]}", rank=int(sys.argv[3]), world_size=2)
r = dist.get_rank(); E = 3
lo, hi = shard.env_range(r, 2, E)
wl = W.make_config(5, n_envs=E, env_offset=lo)
full = W.make_config(5, n_envs=2 * E)
assert np.array_equal(wl.state, full.state[lo:hi]) and np.array_equal(wl.mu, full.mu[lo:hi])
assert np.array_equal(wl.push_fext, full.push_fext[lo:hi]) and np.array_equal(wl.props, full.props[lo:hi])
assert shard.max_over_ranks(10.0 + r) == 11.0 and shard.sum_over_ranks(E) == 2 * E
g = shard.gather_env_results(torch.arange(lo, hi, dtype=torch.int32))
assert g.tolist() == list(range(2 * E))
assert shard.split_envs(7, 2) == [(0, 4), (4, 7)]
dist.destroy_process_group()
print("ok", r)
'''


def test_env_sharding_two_ranks_gloo(tmp_path):
    import socket
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    script = tmp_path / "worker.py"
    script.write_text(_WORKER)
    procs = [subprocess.Popen([sys.executable, str(script), ROOT, str(port), str(r)], stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)
             for r in range(2)]
    outs = [p.communicate(timeout=240)[0] for p in procs]
    assert all(p.returncode == 0 for p in procs), outs


def test_bench_gpus_n_launches_its_own_ranks():
    """`python bench.py --gpus 2` with no launcher re-execs under torch.distributed.run: the dry run
    (gloo, no GPU work) shows two ranks, rank-owned env ranges and the max-over-ranks reduction."""
    import json
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--envs", "64", "--steps", "4", "--dry-run", "--backend", "gloo"],
                         capture_output=True, text=True, timeout=300, env={k: v for k, v in os.environ.items() if k not in ("RANK", "WORLD_SIZE", "LOCAL_RANK")})
    assert out.returncode == 0, out.stderr[-2000:]
    line = [l for l in out.stdout.splitlines() if l.startswith("{")][-1]
    d = json.loads(line)
    assert d["n_gpus"] == 2 and d["total_envs"] == 128 and d["env_ranges_rank0"] == [0, 64] and d["ms_max_over_ranks"] == 101.0
    # without --dry-run the two spawned ranks fail only where the GPU is needed
    import torch
    if not torch.cuda.is_available():
        out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--envs", "64", "--steps", "4"],
                             capture_output=True, text=True, timeout=300, env={k: v for k, v in os.environ.items() if k not in ("RANK", "WORLD_SIZE", "LOCAL_RANK")})
        assert out.returncode != 0 and "bench.py needs a CUDA device" in out.stderr
