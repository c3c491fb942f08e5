"""CPU-only checks: the C-ABI library loads and exports every symbol the header declares, the
binding refuses to run without a GPU (no CPU fallback), and the multi-rank sharding logic
(world_size 2 over gloo)."""
import ctypes
import os
import re
import socket
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _header_functions():
    src = open(os.path.join(ROOT, "include", "berryeasy_b200.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(be_[a-z_0-9]+)\s*\(", src)))


def test_library_builds_and_exports_every_declared_symbol():
    from paper_2312_13051_b200 import build, binding
    path = build.build()
    lib = ctypes.CDLL(path)
    names = _header_functions()
    assert len(names) >= 17
    for n in names:
        assert hasattr(lib, n), f"{n} declared in the header but not exported"
    assert set(binding.EXPORTS) == set(names)
    assert lib.be_strerror is not None
    lib.be_strerror.restype = ctypes.c_char_p
    assert lib.be_strerror(0) == b"ok" and b"NULL" in lib.be_strerror(-1)


def test_argument_checks_need_no_gpu():
    from paper_2312_13051_b200 import build
    lib = ctypes.CDLL(build.build())
    assert lib.be_create(None, None) == -1
    assert lib.be_destroy(None) == -1
    lib.be_workspace_bytes.restype = ctypes.c_size_t
    assert lib.be_workspace_bytes(None, 2, 1) == 0


def test_no_cpu_fallback_without_cuda():
    import torch
    if torch.cuda.is_available():
        pytest.skip("CUDA present")
    from paper_2312_13051_b200.binding import Context
    with pytest.raises(RuntimeError):
        Context()


def test_product_path_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_2312_13051_b200")
    pat = re.compile(r"^\s*(from|import)\s+oracle\b|#include\s+\"[^\"]*oracle", re.M)
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                assert not pat.search(open(os.path.join(dirpath, f)).read()), f


def test_shard_range_partitions():
    from paper_2312_13051_b200.sharding import shard_range
    for n in (0, 1, 7, 24, 4096):
        for w in (1, 2, 3, 8):
            spans = [shard_range(n, r, w) for r in range(w)]
            assert spans[0][0] == 0 and spans[-1][1] == n
            assert all(spans[i][1] == spans[i + 1][0] for i in range(w - 1))
            sizes = [b - a for a, b in spans]
            assert max(sizes) - min(sizes) <= 1


_WORKER = r"""
import os, sys
sys.path.insert(0, {root!r})
import torch, torch.distributed as dist
from paper_2312_13051_b200.sharding import shard_range, gather_phases
dist.init_process_group("gloo", rank=int(os.environ["RANK"]), world_size=int(os.environ["WORLD_SIZE"]))
rank, world = dist.get_rank(), dist.get_world_size()
n_total, m = 7, 3
full = torch.arange(n_total * m, dtype=torch.float64).reshape(n_total, m)
lo, hi = shard_range(n_total, rank, world)
got = gather_phases(full[lo:hi].clone(), n_total, rank, world)
assert torch.equal(got, full), (rank, got)
t = torch.tensor([float(rank + 1)])
dist.all_reduce(t, op=dist.ReduceOp.MAX)      # bench.py's max-over-ranks timing
assert t.item() == world
dist.barrier(); dist.destroy_process_group()
print("OK", rank)
"""


def test_world_size_2_gloo_gather(tmp_path):
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    script = tmp_path / "worker.py"
    script.write_text(_WORKER.format(root=ROOT))
    procs = []
    for r in range(2):
        env = dict(os.environ, RANK=str(r), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.STDOUT, text=True))
    for p in procs:
        out, _ = p.communicate(timeout=180)
        assert p.returncode == 0 and "OK" in out, out
