"""CPU-only checks of the host side: the C-ABI library loads and exports every symbol that
include/rgf.h declares, argument validation that needs no GPU, and the N>1 energy sharding over
torch.distributed (gloo, world_size 2)."""
import ctypes
import os
import re
import subprocess
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_library_exports_every_declared_symbol():
    from paper_1107_5300_b200 import build
    lib = ctypes.CDLL(build.build())
    hdr = open(os.path.join(ROOT, "include", "rgf.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    names = set(re.findall(r"\b(rgf_[a-z0-9_]+)\s*\(", hdr))
    assert {"rgf_plan_create", "rgf_set_device", "rgf_set_device_batch", "rgf_transmission", "rgf_destroy",
            "rgf_last_error"} <= names
    for n in sorted(names):
        assert hasattr(lib, n), n


def test_binding_names_match_header():
    from paper_1107_5300_b200 import binding
    hdr = open(os.path.join(ROOT, "include", "rgf.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    for n in set(re.findall(r"\b(rgf_[a-z0-9_]+)\s*\(", hdr)):
        assert hasattr(binding, n), n


def test_no_gpu_fails_loudly_not_silently():
    """Without a CUDA device plan creation must raise (there is no CPU fallback to fall into)."""
    import torch
    from paper_1107_5300_b200 import binding
    if torch.cuda.is_available():
        return
    try:
        binding.rgf_plan_create(0)
    except binding.RgfError as e:
        assert e.code == binding.RGF_ECUDA
    else:
        raise AssertionError("rgf_plan_create succeeded without a GPU")


def test_product_does_not_import_oracle():
    for root, _, files in os.walk(os.path.join(ROOT, "paper_1107_5300_b200")):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(root, f)).read()
                bad = re.findall(r"import\s+oracle|from\s+oracle|from\s+\.\.?\s*oracle|oracle/|liboracle|rgf_oracle|orc_[a-z_]+\(", src)
                assert not bad, (f, bad, "the product path must not reference oracle/")


def test_shard_roundtrip():
    from paper_1107_5300_b200 import inputs
    E = np.linspace(-1, 1, 13)
    for world in (1, 2, 3, 8):
        parts = [inputs.shard(E, world, r) for r in range(world)]
        assert sum(len(p) for p in parts) == 13
        assert np.array_equal(inputs.unshard(parts, 13), E)


def test_library_shard_helpers_match_the_generator_side():
    """rgf_shard_count / rgf_shard_energies / rgf_unshard (host-only C ABI) against numpy slicing, ragged counts included."""
    from paper_1107_5300_b200 import binding as rgf, inputs
    E = np.linspace(-1, 1, 13)
    for world in (1, 2, 3, 5, 8, 16):
        full = np.full((2, 13), np.nan)
        for r in range(world):
            cnt = rgf.rgf_shard_count(13, world, r)
            assert cnt == len(inputs.shard(E, world, r))
            mine = np.empty(max(cnt, 1))
            assert rgf.rgf_shard_energies(E, 13, world, r, mine) == cnt
            assert np.array_equal(mine[:cnt], inputs.shard(E, world, r))
            part = np.ascontiguousarray(np.stack([mine[:cnt] * 10, mine[:cnt] * 100]))
            if cnt:
                rgf.rgf_unshard(part, 2, 13, world, r, full)
        assert np.array_equal(full, np.stack([E * 10, E * 100]))
    assert rgf.rgf_shard_count(13, 2, 2) == rgf.RGF_EINVAL and rgf.rgf_shard_count(13, 0, 0) == rgf.RGF_EINVAL


_WORKER = r"""
import os, sys
import numpy as np
import torch, torch.distributed as dist
sys.path.insert(0, sys.argv[1])
from paper_1107_5300_b200 import inputs
from oracle import rgf_oracle as orc
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
w = inputs.config0(M=8, L=6, n_E=10)
mine = inputs.shard(w.energies, world, rank)
T = orc.transmission_batch(w.onsite[0], None, w.t, mine, w.eta, nthreads=1)
buf = [torch.zeros(5, dtype=torch.float64) for _ in range(world)]
dist.all_gather(buf, torch.from_numpy(T))
t = torch.tensor([float(rank + 1)], dtype=torch.float64)
dist.all_reduce(t, op=dist.ReduceOp.MAX)          # the bench takes the max time over ranks
if rank == 0:
    full = inputs.unshard([b.numpy() for b in buf], 10)
    ref = orc.transmission_batch(w.onsite[0], None, w.t, w.energies, w.eta, nthreads=1)
    assert np.array_equal(full, ref), (full, ref)
    assert t.item() == world
    print("OK")
dist.destroy_process_group()
"""


def test_energy_sharding_two_ranks_gloo(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(_WORKER)
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2", "--master-addr", "127.0.0.1",
           "--master-port", "29541", str(script), ROOT]
    out = subprocess.run(cmd, capture_output=True, text=True, timeout=300)
    assert out.returncode == 0, out.stderr[-2000:]
    assert "OK" in out.stdout
