"""ptflash_flash_static: the flash for callers that must not allocate GPU memory.

Who they are: a simulator that has handed all device memory to its own arena (or runs under a framework whose caching
allocator has), so that a library's own cudaMalloc can fail; a time-step loop that cannot afford the device-wide stall
of cudaMalloc / cudaFree when the handle's workspace grows; a job held to a fixed memory budget on a shared GPU.  For
them the library carries a fixed 32 MiB workspace inside its device code and one handle-free entry point that uses it
(include/ptflash.h).  What has to hold, and is checked here against the ordinary handle path (ptflash_flash):
  * same answers, call after call, although every call reuses the one array and finds the previous call's queues,
    states and counters in it (also a previous call with another component count, i.e. another carving of the array);
  * a batch beyond PTFLASH_STATIC_MAX_N is refused with a message that names the limit, before anything is launched;
  * the calls do not change the amount of free device memory.

This file sorts after the other test files on purpose: `pytest -x` stops at the first failure, and a failure of this
side entrance should not hide the parity tests of the main path.  It neither needs nor disturbs their state: it passes
alone in a fresh process and at the end of the whole suite."""
import ctypes

import numpy as np
import pytest

from paper_2205_03090_b200 import workloads as W

TOL = 1e-8   # the bar of tests/test_gpu_parity.py for beta, x, y


def _system_args(system):
    import numpy as np
    return (len(system.Tc), np.asarray(system.Tc, float), np.asarray(system.Pc, float), np.asarray(system.omega, float),
            None if system.kij is None else np.asarray(system.kij, float))


def test_static_entry_refuses_what_does_not_fit():
    """The size and argument checks come before the first CUDA call, so they can be exercised without a GPU."""
    from paper_2205_03090_b200 import binding as B, build
    build.build()
    L = B.load_library()
    Tc = (ctypes.c_double * 2)(190.0, 600.0)
    Pc = (ctypes.c_double * 2)(46.0, 21.0)
    om = (ctypes.c_double * 2)(0.01, 0.5)
    one = ctypes.c_void_p(256)   # never dereferenced: every call below is refused first
    args = (one,) * 8 + (None,)
    assert B.STATIC_MAX_N == 32768
    assert L.ptflash_flash_static(2, Tc, Pc, om, None, B.STATIC_MAX_N + 1, *args) == B.PTFLASH_EINVAL
    msg = L.ptflash_last_error().decode()
    assert "PTFLASH_STATIC_MAX_N" in msg and "32768" in msg and "ptflash_flash" in msg
    assert L.ptflash_flash_static(2, Tc, Pc, om, None, 1 << 40, *args) == B.PTFLASH_EINVAL
    assert L.ptflash_flash_static(2, Tc, Pc, om, None, -1, *args) == B.PTFLASH_EINVAL
    assert L.ptflash_flash_static(1, Tc, Pc, om, None, 10, *args) == B.PTFLASH_EINVAL
    assert L.ptflash_flash_static(17, Tc, Pc, om, None, 10, *args) == B.PTFLASH_EINVAL
    assert L.ptflash_flash_static(2, None, Pc, om, None, 10, *args) == B.PTFLASH_EINVAL
    kij = (ctypes.c_double * 4)(0.0, 0.1, 0.2, 0.0)
    assert L.ptflash_flash_static(2, Tc, Pc, om, kij, 10, *args) == B.PTFLASH_EINVAL
    assert "symmetric" in L.ptflash_last_error().decode()
    assert L.ptflash_flash_static(2, Tc, Pc, om, None, 10, None, *args[1:]) == B.PTFLASH_EINVAL   # null z
    assert L.ptflash_flash_static(2, Tc, Pc, om, None, 0, *((None,) * 9)) == B.PTFLASH_OK          # N = 0: no-op


@pytest.mark.gpu
def test_static_entry_matches_the_handle_path_call_after_call():
    import torch
    from paper_2205_03090_b200 import binding as B
    dev = torch.device("cuda:0")
    torch.cuda.set_device(dev)
    # Four batches back to back on one stream, no synchronisation in between, so each call starts on the array exactly
    # as the one before left it: the 10-component system nearly at the size limit, a smaller batch of the same system
    # (the tail of the array still holds the first call's state), the binary system (2 components: the array is carved
    # differently and other kernel instantiations do their first-call set-up), and the large batch again.
    cases = [W.config3(32768 - 91, offset=0), W.config3(5003, offset=500_000), W.config1(1000), W.config3(32768, offset=900_000)]
    f64 = dict(dtype=torch.float64, device=dev)
    i32 = dict(dtype=torch.int32, device=dev)
    ins, outs = [], []
    for w in cases:
        nc, N = w.z.shape
        ins.append(tuple(torch.from_numpy(np.ascontiguousarray(a)).to(dev) for a in (w.z, w.P, w.T)))
        # outputs pre-filled with a pattern no result can equal, so an element the call did not write is seen
        outs.append(dict(beta=torch.full((N,), -7.0, **f64), x=torch.full((nc, N), -7.0, **f64), y=torch.full((nc, N), -7.0, **f64),
                         phase=torch.full((N,), -7, **i32), iters=torch.full((N,), -7, **i32)))
    # the handle path first: its answers are the yardstick, and its allocations are out of the way before memory is watched
    ref = []
    for w, (z, P, T) in zip(cases, ins):
        f = B.PTFlash.from_system(w.system)
        ref.append({k: v.cpu().numpy() for k, v in f.flash(z, P, T, extended=False).items()})
        torch.cuda.synchronize()
        f.close()

    def run(i):
        w, (z, P, T), o = cases[i], ins[i], outs[i]
        nc, Tc, Pc, om, kij = _system_args(w.system)
        B.ptflash_flash_static(nc, Tc, Pc, om, kij, w.N, z, P, T, o["beta"], o["x"], o["y"], o["phase"], o["iters"])

    run(0)                       # first call on this device: also the set-up (see the header), before memory is watched
    run(2)                       # ... and the set-up of the 2-component kernels
    torch.cuda.synchronize()
    for o in (outs[0], outs[2]):
        for k, v in o.items():
            v.fill_(-7)
    torch.cuda.synchronize()
    free_before, _ = torch.cuda.mem_get_info(dev)
    for i in range(len(cases)):
        run(i)
    torch.cuda.synchronize()
    free_after, _ = torch.cuda.mem_get_info(dev)
    assert free_after >= free_before, f"device memory in use grew by {free_before - free_after} bytes over four static calls"

    for i, w in enumerate(cases):
        g = {k: v.cpu().numpy() for k, v in outs[i].items()}
        r = ref[i]
        assert np.array_equal(g["phase"], r["phase"]), f"call {i}: phase labels differ at {np.where(g['phase'] != r['phase'])[0][:5]}"
        assert np.array_equal(g["iters"], r["iters"]), f"call {i}: iteration counts differ"
        assert (g["phase"] == 2).sum() > 0.05 * w.N and (g["phase"] == 1).sum() > 0.05 * w.N   # both branches exercised
        for k in ("beta", "x", "y"):
            assert np.isfinite(g[k]).all()
            err = np.abs(g[k] - r[k]).max()
            assert err <= TOL, f"call {i}: max |static - handle| of {k} = {err:.3e}"
        print(f"static call {i}: nc={w.z.shape[0]} N={w.N} two-phase {(g['phase'] == 2).sum()}, max |beta diff| "
              f"{np.abs(g['beta'] - r['beta']).max():.1e}")

    # refused on the GPU box too, and nothing is written
    w, (z, P, T), o = cases[3], ins[3], outs[3]
    nc, Tc, Pc, om, kij = _system_args(w.system)
    with pytest.raises(B.PTFlashError, match="PTFLASH_STATIC_MAX_N"):
        B.ptflash_flash_static(nc, Tc, Pc, om, kij, B.STATIC_MAX_N + 1, z, P, T, o["beta"], o["x"], o["y"], o["phase"], o["iters"])
