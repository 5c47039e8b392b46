"""CPU-only checks of the boundary and the host logic: the C-ABI library loads and exports every symbol
include/ptflash.h declares (no compute calls without a GPU); argument validation that needs no device;
the multi-GPU sharding recipe of bench.py under gloo with world_size 2."""
import ctypes
import os
import re
import subprocess
import sys
from pathlib import Path

import numpy as np
import pytest

ROOT = Path(__file__).resolve().parents[1]


@pytest.fixture(scope="module")
def lib():
    from paper_2205_03090_b200 import build as B, binding
    B.build()
    return binding.load_library()


def test_abi_exports_every_declared_symbol(lib):
    hdr = (ROOT / "include" / "ptflash.h").read_text()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(ptflash_[a-z0-9_]+)\s*\(", hdr))
    assert {"ptflash_create", "ptflash_flash", "ptflash_destroy", "ptflash_flash_ex", "ptflash_flash_host"} <= declared
    for name in declared:
        assert hasattr(lib, name), f"{name} declared in include/ptflash.h but not exported"
    from paper_2205_03090_b200 import binding
    assert set(binding.EXPORTS) == declared
    assert b"sm_100a" in lib.ptflash_version()


def test_sass_is_sm100a(lib):
    so = ROOT / "paper_2205_03090_b200" / "libptflash.so"
    out = subprocess.run(["cuobjdump", "-lelf", str(so)], capture_output=True, text=True).stdout
    assert "sm_100a" in out


def test_create_validation_without_gpu(lib):
    # argument errors are detected before any CUDA call
    Tc = (ctypes.c_double * 2)(190.0, 600.0)
    Pc = (ctypes.c_double * 2)(46.0, 21.0)
    om = (ctypes.c_double * 2)(0.01, 0.5)
    assert not lib.ptflash_create(1, Tc, Pc, om, None)
    assert b"nc" in lib.ptflash_last_error()
    assert not lib.ptflash_create(17, Tc, Pc, om, None)
    assert not lib.ptflash_create(2, None, Pc, om, None)
    bad = (ctypes.c_double * 2)(-1.0, 600.0)
    assert not lib.ptflash_create(2, bad, Pc, om, None)
    kij = (ctypes.c_double * 4)(0.0, 0.1, 0.2, 0.0)
    assert not lib.ptflash_create(2, Tc, Pc, om, kij)
    assert b"symmetric" in lib.ptflash_last_error()
    # null handle
    assert lib.ptflash_flash(None, 10, None, None, None, None, None, None, None, None, None) == -1
    assert lib.ptflash_destroy(None) == 0
    assert lib.ptflash_set_option(None, 0, 1.0) == -1


def test_binding_fails_loudly_without_library(tmp_path, monkeypatch):
    from paper_2205_03090_b200 import binding
    monkeypatch.setattr(binding, "_lib", None)
    monkeypatch.setattr(binding, "_LIB_PATH", tmp_path / "missing.so")
    with pytest.raises(binding.PTFlashError):
        binding.ptflash_version()


def test_product_does_not_import_oracle():
    for p in (ROOT / "paper_2205_03090_b200").rglob("*"):
        if p.suffix in (".py", ".cu", ".cuh", ".h") and p.is_file():
            txt = p.read_text()
            assert "import oracle" not in txt and "from oracle" not in txt and "ptflash_oracle" not in txt, p


_WORKER = r"""
import os, sys, time
sys.path.insert(0, {root!r})
import numpy as np, torch, torch.distributed as dist
from paper_2205_03090_b200 import workloads as W
from oracle.oracle import Oracle
dist.init_process_group("gloo", init_method="tcp://127.0.0.1:{port}", rank=int(sys.argv[1]), world_size=2)
rank, world = dist.get_rank(), dist.get_world_size()
N = 600
w = W.config3(N, offset=rank * N)            # bench.py's sharding recipe: disjoint counter ranges per rank
t0 = time.perf_counter()
r = Oracle.from_system(w.system).flash(w.z, w.P, w.T, nthreads=1)
dt = torch.tensor([time.perf_counter() - t0], dtype=torch.float64)
dist.barrier()
dist.all_reduce(dt, op=dist.ReduceOp.MAX)     # max-over-ranks timing
two = torch.tensor([float((r["phase"] == 2).sum())], dtype=torch.float64)
dist.all_reduce(two)
beta = [torch.zeros(N, dtype=torch.float64) for _ in range(world)]
dist.all_gather(beta, torch.from_numpy(np.nan_to_num(r["beta"])))
if rank == 0:
    full = W.config3(world * N)
    rf = Oracle.from_system(full.system).flash(full.z, full.P, full.T, nthreads=1)
    assert np.array_equal(np.concatenate([b.numpy() for b in beta]), np.nan_to_num(rf["beta"]))
    assert int(two.item()) == int((rf["phase"] == 2).sum())
    assert dt.item() > 0
    print("OK", world * N / dt.item())
dist.destroy_process_group()
"""


def test_sharding_world_size_2_gloo(tmp_path, oracle_mod):
    port = 29500 + (os.getpid() % 400)
    script = tmp_path / "worker.py"
    script.write_text(_WORKER.format(root=str(ROOT), port=port))
    procs = [subprocess.Popen([sys.executable, str(script), str(r)], stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True)
             for r in range(2)]
    outs = [p.communicate(timeout=300) for p in procs]
    for p, (o, e) in zip(procs, outs):
        assert p.returncode == 0, e[-2000:]
    assert "OK" in outs[0][0]
