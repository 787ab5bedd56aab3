"""CPU-only: the C-ABI library loads and exports every symbol include/west.h declares (no compute without a GPU),
the binding fails loudly instead of falling back, and the bench's rank/shard arithmetic is right (gloo, world_size 2)."""
import ctypes as C
import os
import re
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _ensure_built():
    from paper_2203_05623_b200 import build as b
    b.build(force=False)


def test_library_exports_every_declared_symbol():
    _ensure_built()
    import paper_2203_05623_b200 as wb
    hdr = open(os.path.join(ROOT, "include", "west.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = sorted(set(re.findall(r"\b(west_[a-z0-9_]+)\s*\(", hdr)))
    assert len(declared) >= 15
    lib = C.CDLL(wb.LIB_PATH)
    for name in declared:
        assert hasattr(lib, name), "missing export " + name
    assert sorted(wb.EXPORTS) == declared, "binding.EXPORTS and west.h disagree"


def test_no_cpu_fallback_without_a_device():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    _ensure_built()
    import paper_2203_05623_b200 as wb
    lib = wb.load_library()
    ctx = C.c_void_p()
    cell = wb.west_cell(10.0, 25, 24, wb.WEST_FULL)
    rc = lib.west_create(C.byref(ctx), C.byref(cell), None)
    assert rc == wb.binding.WEST_ECUDA
    assert b"no CPU fallback" in lib.west_last_error(None)
    bad = wb.west_cell(10.0, 25, 25, wb.WEST_FULL)
    assert lib.west_create(C.byref(ctx), C.byref(bad), None) == wb.binding.WEST_EINVAL


def test_binding_raises_when_library_is_missing(tmp_path, monkeypatch):
    import paper_2203_05623_b200.binding as b
    monkeypatch.setattr(b, "LIB_PATH", str(tmp_path / "libwest.so"))
    with pytest.raises(ImportError):
        b.load_library()


def test_product_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_2203_05623_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".hpp")):
                src = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in src, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith(".py"):
            assert "paper_2203_05623_b200" not in open(os.path.join(ROOT, "oracle", f)).read().replace(
                "``paper_2203_05623_b200/``", "")


_WORKER = r"""
import os, sys
sys.path.insert(0, %r)
import numpy as np, torch, torch.distributed as dist
import synth
dist.init_process_group("gloo", rank=int(os.environ["RANK"]), world_size=int(os.environ["WORLD_SIZE"]))
rank, world = dist.get_rank(), dist.get_world_size()
cfg = synth.get_config("cfg1")
n_pert = 2
# the bench's sharding rule: rank r owns perturbation streams [r*n_pert, (r+1)*n_pert)
mine = synth.perturbations(cfg, n_pert=n_pert, first=rank * n_pert)
allp = synth.perturbations(cfg, n_pert=n_pert * world, first=0)
assert np.array_equal(mine, allp[rank * n_pert:(rank + 1) * n_pert])
# the bench's timing rule: max over ranks
t = torch.tensor([10.0 + rank, 1.0], dtype=torch.float64)
dist.all_reduce(t, op=dist.ReduceOp.MAX)
assert float(t[0]) == 10.0 + world - 1
dist.barrier()
if rank == 0:
    print("OK", world)
dist.destroy_process_group()
"""


def test_perturbation_sharding_world_size_2_gloo(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(_WORKER % ROOT)
    env = dict(os.environ, MASTER_ADDR="127.0.0.1", MASTER_PORT="29653", WORLD_SIZE="2")
    procs = [subprocess.Popen([sys.executable, str(script)], env=dict(env, RANK=str(r)), stdout=subprocess.PIPE, stderr=subprocess.PIPE,
                              text=True) for r in range(2)]
    outs = [p.communicate(timeout=180) for p in procs]
    for p, (o, e) in zip(procs, outs):
        assert p.returncode == 0, e
    assert "OK 2" in outs[0][0]
