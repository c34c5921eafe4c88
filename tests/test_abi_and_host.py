"""-m "not gpu": the C-ABI library loads and exports every symbol include/bathy.h declares, argument
errors are reported without touching a device, and the N > 1 host logic works under gloo."""
import ctypes as C
import os
import re
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "bathy.h")


def _declared():
    src = open(HEADER).read()
    names = re.findall(r"BATHY_API\s+[\w\s\*]+?\b(\w+)\s*\(", src)
    assert len(names) >= 13
    return names


@pytest.fixture(scope="module")
def shared_lib():
    from paper_2505_22675_b200 import build
    return C.CDLL(build.build())


def test_every_declared_symbol_is_exported(shared_lib):
    from paper_2505_22675_b200 import binding
    for name in _declared():
        assert hasattr(shared_lib, name), f"{name} declared in include/bathy.h but not exported"
    assert sorted(binding.SYMBOLS) == sorted(_declared())


def test_no_torch_or_cxx_types_in_the_header():
    src = open(HEADER).read()
    assert 'extern "C"' in src
    code = re.sub(r"/\*.*?\*/", "", src, flags=re.S)                     # comments may mention cudaStream_t
    for banned in ("torch", "at::", "std::", "Tensor", "cudaStream_t", "#include <cuda"):
        assert banned not in code


def test_only_declared_symbols_are_visible():
    from paper_2505_22675_b200 import build
    out = subprocess.run(["nm", "-D", "--defined-only", build.build()], capture_output=True, text=True).stdout
    exported = {l.split()[-1] for l in out.splitlines() if " T " in l}
    assert set(_declared()) <= exported
    assert not any(s.startswith("_ZN5bathy") for s in exported), "internal C++ symbols leak from libbathy.so"


def test_strerror_and_argument_errors_need_no_device():
    import paper_2505_22675_b200 as b
    L = b.lib()
    assert L.bathy_strerror(0) and L.bathy_strerror(-3) and L.bathy_strerror(-12345)
    g = b.binding.GridGeom(4, 4, 0.0, 0.0, 1.0, 1.0)
    bad = b.binding.GridGeom(1, 4, 0.0, 0.0, 1.0, 1.0)
    assert L.interp_bilinear(None, g, None, g, None) == -1                 # BATHY_ERR_NULL
    assert L.interp_bilinear(C.c_void_p(16), bad, C.c_void_p(32), g, None) == -2   # BATHY_ERR_GEOMETRY
    assert L.interp_spline(C.c_void_p(16), g, C.c_void_p(32), g, None, 0, None) in (-5, -1)
    v = b.binding.Variogram(0, 1.0, 1.0, 0.0)
    assert L.krige_predict(None, g, v, 4, C.c_void_p(16), None, None, None) == -8  # BATHY_ERR_INDEX
    assert L.bathy_launch_count() >= 0


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_2505_22675_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", text, re.M), f
                assert "oracle.c" not in text and "liboracle" not in text, f


def test_sharding_helpers():
    from paper_2505_22675_b200 import sharding as S
    assert S.rank_seed(1004, 0) == 1004 and S.rank_seed(1004, 3) == 1304
    assert [S.tile_owner(t, 4) for t in range(6)] == [0, 1, 2, 3, 0, 1]
    tiles = list(range(64))
    parts = [S.tiles_of_rank(tiles, r, 8) for r in range(8)]
    assert sorted(sum(parts, [])) == tiles and all(len(p) == 8 for p in parts)
    assert S.whole_job_throughput(1000.0, 4, 2.0) == 2.0e6
    assert S.reduce_step_times([1.0, 2.0]) == [1.0, 2.0]


_WORKER = r'''
import os, sys
sys.path.insert(0, sys.argv[1])
import torch.distributed as dist
from paper_2505_22675_b200 import sharding as S, workloads as W
dist.init_process_group("gloo", init_method="tcp://127.0.0.1:" + sys.argv[2], rank=int(sys.argv[3]), world_size=2)
rank = dist.get_rank()
w = W.sounding_config(4, width=60.0, n_target=900, n_out=16, seed=S.rank_seed(W.SEEDS[4], rank))
ms = S.reduce_step_times([10.0 + 5.0 * rank, 3.0 - rank], dist)            # max over ranks, entry by entry
import torch
chk = torch.tensor([float(w.x.sum())], dtype=torch.float64)
gathered = [torch.zeros_like(chk) for _ in range(2)]
dist.all_gather(gathered, chk)
# one-survey sharding (NEXT-4): rank 0's soundings are replicated, the tiles are dealt round-robin
w0 = W.sounding_config(5, width=60.0, n_target=900, n_out=32, seed=W.SEEDS[5])
xs = [torch.from_numpy(a.copy()) if rank == 0 else torch.zeros(a.shape[0]) for a in (w0.x, w0.y, w0.z)]
S.broadcast_soundings(*xs, dist, 0)
assert all(torch.equal(t, torch.from_numpy(a)) for t, a in zip(xs, (w0.x, w0.y, w0.z)))
tiles = W.boustrophedon_tiles(32, 8)
mine = S.tiles_of_rank(tiles, rank, 2)
cnt = torch.tensor([float(len(mine)), float(sum(t[2] * t[3] for t in mine))], dtype=torch.float64)
dist.all_reduce(cnt)
assert cnt.tolist() == [16.0, 1024.0], cnt
dist.barrier()
if rank == 0:
    assert ms == [15.0, 3.0], ms
    assert gathered[0].item() != gathered[1].item()                   # the two ranks drew different batches
    print("value", S.whole_job_throughput(w.geom_out.n, 2, ms[0]))
dist.destroy_process_group()
'''


def test_two_ranks_gloo(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(_WORKER)
    port = str(29500 + os.getpid() % 2000)
    procs = [subprocess.Popen([sys.executable, str(script), ROOT, port, str(r)], stdout=subprocess.PIPE,
                              stderr=subprocess.STDOUT, text=True) for r in range(2)]
    outs = [p.communicate(timeout=180)[0] for p in procs]
    assert all(p.returncode == 0 for p in procs), outs
    assert "value" in outs[0] and abs(float(outs[0].split("value")[1]) - 2 * 256 / 15e-3) < 1e-6
