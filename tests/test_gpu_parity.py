"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element, on the same
seeded inputs.  Bar (BASELINE.json north_star): phase labels identical except mixtures whose minimum TPD
lies within 1e-9 of zero (reported); beta, x, y within 1e-8 absolute."""
import numpy as np
import pytest

from paper_2205_03090_b200 import workloads as W

pytestmark = pytest.mark.gpu
import os
import sys
sys.path.insert(0, os.path.dirname(__file__))

TOL = 1e-8


def _gpu_flash(w, engine, lnK0=None, flags=None, **opts):
    import torch
    from paper_2205_03090_b200 import binding as B
    dev = torch.device("cuda:0")
    f = B.PTFlash.from_system(w.system, engine=engine, **opts)
    z, P, T = (torch.from_numpy(a).to(dev) for a in (w.z, w.P, w.T))
    l0 = torch.from_numpy(np.ascontiguousarray(lnK0)).to(dev) if lnK0 is not None else None
    fl = torch.from_numpy(np.ascontiguousarray(flags, dtype=np.uint8)).to(dev) if flags is not None else None
    out = f.flash(z, P, T, lnK0=l0, flags=fl)
    torch.cuda.synchronize()
    res = {k: v.cpu().numpy() for k, v in out.items()}
    res["stats"] = f.stats()
    f.close()
    return res


def compare(w, g, o, tol=TOL, excuse=None):
    """Element-by-element comparison; returns a report dict.  The near-zero-TPD band (reading C9) is decided from the
    ORACLE's minimum TPD alone: a label mismatch is excused only where the oracle itself reports 0 < |tpd_min| < 1e-9.
    `excuse`: boolean mask of mixtures left out of the comparison (the caller bounds and reports them)."""
    N = w.N
    keep = np.ones(N, dtype=bool) if excuse is None else ~excuse
    mism = np.where((g["phase"] != o["phase"]) & keep)[0]
    in_band = np.isfinite(o["tpd_min"]) & (o["tpd_min"] != 0.0) & (np.abs(o["tpd_min"]) < 1e-9)
    band = mism[in_band[mism]]
    hard = np.setdiff1d(mism, band)
    same2 = (g["phase"] == 2) & (o["phase"] == 2) & keep
    same1 = (g["phase"] == 1) & (o["phase"] == 1) & keep
    db = np.abs(g["beta"] - o["beta"])
    dx = np.abs(g["x"] - o["x"]).max(0)
    dy = np.abs(g["y"] - o["y"]).max(0)
    err2 = np.maximum(db, np.maximum(dx, dy))
    rep = dict(N=N, two_phase=int(same2.sum()), label_mismatch=len(mism), in_band=len(band),
               oracle_band_size=int(in_band.sum()),
               max_err_two_phase=float(err2[same2].max()) if same2.any() else 0.0,
               max_err_single=float(np.maximum(dx, dy)[same1].max()) if same1.any() else 0.0,
               beta_convention_mismatch=int((db[same1] != 0).sum()))
    msg = []
    for n in hard[:10]:
        msg.append(f"label mismatch n={n} gpu={g['phase'][n]} oracle={o['phase'][n]} tpd_o={o['tpd_min'][n]:.3e} "
                   f"tpd_g={g['tpd_min'][n]:.3e} st_o={o['status'][n]} st_g={g['status'][n]} P={w.P[n]:.3f} T={w.T[n]:.3f}")
    bad = np.where(same2 & (err2 > tol))[0]
    for n in bad[:10]:
        msg.append(f"value mismatch n={n} err={err2[n]:.3e} beta_g={g['beta'][n]:.12f} beta_o={o['beta'][n]:.12f} "
                   f"dc={o['diag'][1, n]:.3e} rate={o['diag'][2, n]:.4f} st_o={o['status'][n]} st_g={g['status'][n]}")
    rep["messages"] = msg
    rep["n_hard"] = len(hard)
    rep["n_bad"] = len(bad)
    rep["bad"] = bad
    rep["band"] = band
    return rep


MAX_BAND_PER_MILLION = 5     # label mismatches excused by the oracle's |tpd_min| < 1e-9 band: listed, and bounded by this


def check(w, g, o, excuse=None):
    rep = compare(w, g, o, excuse=excuse)
    print({k: v for k, v in rep.items() if k not in ("messages", "bad", "band")})
    for n in rep["band"]:
        print(f"  in-band label mismatch n={n}: tpd_min oracle {o['tpd_min'][n]:.3e} gpu {g['tpd_min'][n]:.3e}")
    assert rep["n_hard"] == 0 and rep["n_bad"] == 0, "\n".join(rep["messages"])
    assert rep["in_band"] <= max(1, int(np.ceil(MAX_BAND_PER_MILLION * w.N / 1e6)))
    assert rep["max_err_single"] == 0.0            # single phase: x = y = z bit-exact
    assert rep["beta_convention_mismatch"] == 0
    return rep


def _vec(r, n):
    return np.concatenate([[r["beta"][n]], r["x"][:, n], r["y"][:, n]])


def adjudicate(oracle_mod, w, g, o, idx, lnK0=None, flags=None):
    """Conditioning note of SURVEY.md section 8(c): every two-phase mixture whose beta, x or y differs from the (double)
    oracle by more than 1e-8 is re-flashed by the oracle in long double with tight tolerances -- the best available
    value of the exact fixed point -- and reported with d_c = ||ln K||_2 (eq. 14), the last SS rate and the
    iteration counts.  With e_gpu, e_oracle the distances of the CUDA result and of the double oracle from that value, the
    miss is attributed
      * to the ORACLE's rounding        if e_gpu <= 1e-8 (the CUDA result is within the bar of the exact answer);
      * to CONDITIONING                 if e_gpu <= 4 e_oracle: next to a critical point or the phase boundary the Hessian
        of G is nearly singular and plain fp64 evaluation of ln phi does not fix n^V to 1e-8 -- the double oracle itself
        misses the exact answer by e_oracle > 2.5e-9, and the CUDA path is within a small factor of that;
      * to a BUG                        otherwise (the test fails)."""
    ld = oracle_mod.Oracle.from_system(w.system, real="long double")
    tight = dict(tol_ss=1e-13, tol_newton_g=1e-15, tol_newton_step=1e-13)
    rows = []
    for n in idx:
        z, P, T = np.ascontiguousarray(w.z[:, n:n + 1]), w.P[n:n + 1].copy(), w.T[n:n + 1].copy()
        kw = {} if lnK0 is None else dict(lnK0=np.ascontiguousarray(lnK0[:, n:n + 1]), flags=flags[n:n + 1].copy())
        b = ld.flash(z, P, T, nthreads=1, opts=tight, **kw)
        vg, vo = _vec(g, n), _vec(o, n)
        two = b["phase"][0] == 2
        e_g = float(np.abs(vg - _vec(b, 0)).max()) if two else float("inf")
        e_o = float(np.abs(vo - _vec(b, 0)).max()) if two else float("inf")
        why = "oracle rounding" if e_g <= TOL else ("conditioning" if e_g <= 4.0 * e_o else "BUG")
        rows.append(dict(n=int(n), gap_gpu_oracle=float(np.abs(vg - vo).max()), e_gpu=e_g, e_oracle=e_o, attributed=why,
                         d_c=float(o["diag"][1, n]), ss_rate=float(o["diag"][2, n]), iters_oracle=int(o["iters"][n]),
                         iters_gpu=int(g["iters"][n]), beta_gpu=float(g["beta"][n]), beta_oracle=float(o["beta"][n]),
                         beta_long_double_tight=float(b["beta"][0])))
    return rows


@pytest.mark.parametrize("engine", [0, 1])
@pytest.mark.parametrize("cfg,N", [(1, 1000), (2, 20000), (3, 20000), (4, 20000)])
def test_parity_configs(oracle_mod, cfg, N, engine):
    w = W.CONFIGS[cfg](N)
    o = oracle_mod.Oracle.from_system(w.system).flash(w.z, w.P, w.T)
    g = _gpu_flash(w, engine)
    rep = check(w, g, o)
    assert rep["two_phase"] > 0.05 * N
    # iteration counts are path-dependent but should agree on almost all mixtures
    assert (g["iters"] == o["iters"]).mean() > 0.98


def test_parity_config5_warm_start(oracle_mod):
    """BASELINE config 5: caller-supplied lnK0 near the phase boundary + skip-stability flags (warm) vs Wilson (cold)."""
    import config5
    orc = oracle_mod.Oracle.from_system(W.system_co2_10())
    w, lnK0, flags, info = config5.build(orc, 6000)
    o_warm = orc.flash(w.z, w.P, w.T, lnK0=lnK0, flags=flags)
    o_cold = info["cold"]
    for engine in (1, 0):
        g_warm = _gpu_flash(w, engine, lnK0=lnK0, flags=flags)
        g_cold = _gpu_flash(w, engine)
        rep_w = check(w, g_warm, o_warm)
        rep_c = check(w, g_cold, o_cold)
        two = (g_warm["phase"] == 2) & (g_cold["phase"] == 2)
        assert two.sum() > 2000
        # warm and cold starts reach the same split wherever both report two phases, liquid/vapour labels included:
        # the identity no longer follows the sign of the supplied lnK0 but the compressibility factors (reading C23)
        db = np.abs(g_warm["beta"] - g_cold["beta"])[two]
        assert np.all(db < 1e-8)
        restarted = (g_warm["status"] & 64) != 0
        assert np.all(g_warm["stab_iters"][(flags == 1) & ~restarted] == 0)   # stability skipped where the caller said so
        # a failed skip-stability hint is dropped and reported (ST_WARM_RESTART), on both sides for the same mixtures
        # up to a handful of borderline cases; after the restart the answer is the cold one
        assert 0 < restarted.sum() < 0.03 * w.N
        # both sides drop a hinted split that is still outside 0 < theta < 1 after 12 SS iterations or unconverged after 15
        # trust-region iterations (C21).  With the oracle's restricted step (PTFLASH_OPT_HINT_ETA_SEARCH = 1) they restart the
        # same mixtures up to a handful of borderline cases; the default (the truncated modified-Cholesky step of C25 for
        # hinted splits too) reaches the same answers but fails / survives on a slightly different set of hints
        o_restarted = (o_warm["status"] & 64) != 0
        assert np.sum(o_restarted != restarted) <= 0.01 * w.N
        if engine == 1:
            g_eta = _gpu_flash(w, engine, lnK0=lnK0, flags=flags, hint_eta_search=1)
            check(w, g_eta, o_warm)
            assert np.sum(o_restarted != ((g_eta["status"] & 64) != 0)) <= 3
            # the early start of the probe-found splits (scheduling only) also after a hinted pre-pass: identical bits
            g_early = _gpu_flash(w, engine, lnK0=lnK0, flags=flags, early_split_ss=1)
            for k in ("phase", "beta", "x", "y", "iters", "status"):
                assert np.array_equal(g_early[k], g_warm[k]), k
        else:
            assert np.sum(o_restarted != restarted) <= 3          # engine 0 follows the oracle's path
        assert np.array_equal(g_warm["phase"][restarted], g_cold["phase"][restarted])
        print("config5 engine", engine, "mean iters (two-phase): warm %.2f cold %.2f; cold stability iters %.2f" %
              (g_warm["iters"][two].mean(), g_cold["iters"][two].mean(), g_cold["stab_iters"][two].mean()), rep_w, rep_c)


@pytest.mark.parametrize("N", [0, 1, 31, 33, 127, 1025])
def test_ragged_sizes(oracle_mod, N):
    import torch
    from paper_2205_03090_b200 import binding as B
    w = W.config3(max(N, 1))
    if N == 0:
        f = B.PTFlash.from_system(w.system)
        dev = torch.device("cuda:0")
        e = torch.empty(0, dtype=torch.float64, device=dev)
        B.ptflash_flash(f.h, 0, e, e, e, e, e, e, torch.empty(0, dtype=torch.int32, device=dev))   # no-op
        f.close()
        return
    o = oracle_mod.Oracle.from_system(w.system).flash(w.z, w.P, w.T)
    for engine in (1, 0):
        check(w, _gpu_flash(w, engine), o)


def test_invalid_and_degenerate_inputs(oracle_mod):
    """O0 validation, z_i = 0 components (C12), unnormalised-within-1e-9 feeds (C20)."""
    w = W.config3(64)
    z, P, T = w.z.copy(), w.P.copy(), w.T.copy()
    z[:, 1] = np.nan
    P[2] = -5.0
    T[3] = 0.0
    z[0, 4] = -1e-3
    z[:, 5] *= 1.001                       # sum z = 1.001 -> invalid
    P[6] = np.inf
    z[:, 7] *= 1.0 + 5e-10                 # within 1e-9 -> valid, normalised internally
    z[2, 8] = 0.0; z[:, 8] /= z[:, 8].sum()  # an absent component
    z[[0, 1, 2, 3, 4, 5, 6, 7], 9] = 0.0; z[:, 9] /= z[:, 9].sum()   # CO2/N2 binary inside the 10-component system
    w2 = W.Workload("edge", w.system, P, T, np.ascontiguousarray(z))
    o = oracle_mod.Oracle.from_system(w.system).flash(w2.z, w2.P, w2.T)
    assert list(o["phase"][1:7]) == [-1] * 6 and o["phase"][7] in (1, 2)
    for engine in (1, 0):
        g = _gpu_flash(w2, engine)
        assert np.array_equal(g["phase"], o["phase"])
        bad = o["phase"] == -1
        assert np.all(np.isnan(g["beta"][bad])) and np.all(np.isnan(g["x"][:, bad])) and np.all(np.isnan(g["y"][:, bad]))
        ok = ~bad
        np.testing.assert_allclose(g["beta"][ok], o["beta"][ok], atol=TOL)
        np.testing.assert_allclose(g["x"][:, ok], o["x"][:, ok], atol=TOL)
        np.testing.assert_allclose(g["y"][:, ok], o["y"][:, ok], atol=TOL)
        assert np.all(g["x"][2, 8] == 0) and np.all(g["y"][2, 8] == 0)
        if engine == 1:
            assert g["stats"]["n_invalid"] == 6


def _system_16(nc):
    """Up to 16 components: the CO2-rich ten plus six alkanes duplicated with perturbed constants, truncated to nc."""
    s10 = W.system_co2_10()
    Tc = np.concatenate([s10.Tc, s10.Tc[2:8] * 1.03]); Pc = np.concatenate([s10.Pc, s10.Pc[2:8] * 0.97])
    om = np.concatenate([s10.omega, s10.omega[2:8] + 0.01])
    kij = np.zeros((16, 16)); kij[:10, :10] = s10.kij
    kij[10:, 8] = kij[8, 10:] = 0.12; kij[10:, 9] = kij[9, 10:] = 0.10
    return W.System([f"c{i}" for i in range(nc)], Tc[:nc], Pc[:nc], om[:nc], np.ascontiguousarray(kij[:nc, :nc]))


@pytest.mark.parametrize("nc", [3, 13, 16])
def test_other_component_counts(oracle_mod, nc):
    """nc = 3, 13 and 16 (the largest supported): every component count runs the register-resident stage kernels of
    engine 1 (14 launches per call: k_init, k2_probe, k2_stab_ss, k3_stab_newton, k_stab_decide, 4 x k2_split_ss,
    4 x k3_split_newton, k_finalize_counters); for nc >= 13 the Newton CTAs are sized by shared memory."""
    system = W.make_system(["C1", "C3", "nC10"]) if nc == 3 else _system_16(nc)
    N = 3000
    n = np.arange(N)
    T = 220.0 + 300.0 * W.uniform(77, n, 0)
    P = 2.0 + 200.0 * W.uniform(77, n, 1)
    z = W._dirichlet1(77, n, nc)
    w = W.Workload("nc%d" % nc, system, P, T, np.ascontiguousarray(z))
    o = oracle_mod.Oracle.from_system(system).flash(w.z, w.P, w.T)
    for engine in (1, 0):
        g = _gpu_flash(w, engine)
        rep = check(w, g, o)
        assert rep["two_phase"] > 100
        if engine == 1:
            assert g["stats"]["kernel_launches"] == 14 and g["stats"]["n_stab_newton"] > 0 and g["stats"]["n_split_newton"] > 0


@pytest.mark.parametrize("cfg,N", [(1, 600), (3, 1500)])
def test_pure_successive_substitution_mode(oracle_mod, cfg, N):
    """use_newton = 0: every stage runs plain successive substitution (the north_star's SSI path) on the same
    register-resident stage kernels; the Newton stages find empty queues."""
    w = W.CONFIGS[cfg](N)
    opts = dict(use_newton=0, ss_cap=100000)
    o = oracle_mod.Oracle.from_system(w.system).flash(w.z, w.P, w.T, opts=opts)
    for engine in (1, 0):
        g = _gpu_flash(w, engine, **opts)
        check(w, g, o)
        if engine == 1:
            assert g["stats"]["n_stab_newton"] == 0 and g["stats"]["n_split_newton"] == 0


def _paper9_with_crawlers(n_ordinary=3000):
    """The first n_ordinary mixtures of the paper's 9-component workload with the eight "crawlers" of its first 10^6 mixtures
    (tests/golden/paper9_crawlers.json, inputs only, written by tests/golden/make_paper9_crawlers.py) spread among them."""
    import json
    g = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "paper9_crawlers.json")))
    base = W.paper9(n_ordinary)
    P = np.array([float.fromhex(v) for v in g["P"]]); T = np.array([float.fromhex(v) for v in g["T"]])
    z = np.array([[float.fromhex(v) for v in col] for col in g["z"]]).T          # [9, 8]
    pos = np.linspace(17, n_ordinary - 17, len(P)).astype(int)                    # different warps and CTAs
    Pn, Tn, zn = base.P.copy(), base.T.copy(), base.z.copy()
    Pn[pos], Tn[pos], zn[:, pos] = P, T, z
    return W.Workload("paper9_with_crawlers", base.system, Pn, Tn, np.ascontiguousarray(zn)), pos, g["oracle_split_ss_iters"]


def test_split_crawlers_and_early_split_ss(oracle_mod):
    """Splits still outside 0 < theta < 1 when the switch to the Newton stage is due continue the successive substitution
    (reading C13) on the crawler stream (split parts 2 / 3, resumed from the saved iterate): same answers and the same
    iteration counts as the oracle, whichever stream order is used (PTFLASH_OPT_EARLY_SPLIT_SS, with and without the fork)."""
    w, pos, ss_iters = _paper9_with_crawlers()
    o = oracle_mod.Oracle.from_system(w.system).flash(w.z, w.P, w.T)
    assert sorted(int(v) for v in o["stage"][5][pos]) == sorted(ss_iters) and max(ss_iters) > 400
    ref = None
    for opts in (dict(), dict(early_split_ss=1), dict(stage_profile=1)):
        g = _gpu_flash(w, 1, **opts)
        check(w, g, o)
        # iteration counts: probe + SS + Newton updates.  The SS part is the oracle's to the iteration (a crawler that ends
        # inside the SS stage matches exactly); the Newton part takes the truncated step of C25 instead of the eta search
        in_ss = o["stage"][6][pos] == 0
        assert in_ss.any() and np.array_equal(g["iters"][pos][in_ss], o["iters"][pos][in_ss])
        assert np.abs(g["iters"][pos] - o["iters"][pos]).max() <= 8
        assert g["stats"]["max_split_ss_iters"] == max(ss_iters) and g["stats"]["kernel_launches"] == 14
        assert g["stats"]["n_split_newton"] == int(o["stage"][8].sum())          # crawlers that reach the Newton stage are counted
        if ref is None:
            ref = g
        else:
            for k in ("beta", "x", "y", "phase", "iters", "status"):
                assert np.array_equal(g[k], ref[k]), k


def test_host_buffers_stream_and_stats(oracle_mod):
    import torch
    from paper_2205_03090_b200 import binding as B
    w = W.config3(5000)
    dev = torch.device("cuda:0")
    f = B.PTFlash.from_system(w.system)
    z, P, T = (torch.from_numpy(a).to(dev) for a in (w.z, w.P, w.T))
    st = torch.cuda.Stream()
    with torch.cuda.stream(st):
        out = f.flash(z, P, T)                      # enqueued on a non-default stream
    st.synchronize()
    stats = f.stats()
    assert stats["n_total"] == 5000 and stats["kernel_launches"] >= 1
    assert stats["n_probe_case1"] + stats["n_probe_case2"] + stats["n_probe_case3"] + stats["n_invalid"] == 5000
    assert stats["n_two_phase"] == int((out["phase"] == 2).sum())
    assert stats["n_split"] >= stats["n_two_phase"] and stats["n_stability"] == stats["n_probe_case1"] + stats["n_probe_case2"]
    # end-to-end variant with host buffers gives the same bits
    hb = np.empty(5000); hx = np.empty((10, 5000)); hy = np.empty((10, 5000))
    hp = np.empty(5000, dtype=np.int32); hi = np.empty(5000, dtype=np.int32)
    B.ptflash_flash_host(f.h, 5000, w.z, w.P, w.T, hb, hx, hy, hp, hi)
    assert np.array_equal(hp, out["phase"].cpu().numpy()) and np.array_equal(hb, out["beta"].cpu().numpy())
    assert np.array_equal(hx, out["x"].cpu().numpy()) and np.array_equal(hi, out["iters"].cpu().numpy())
    f.close()


def test_two_streams_equal_one_stream(oracle_mod):
    """Engine 1 forks the two parts of the phase split onto two streams after the stability stages; with stage profiling on
    everything runs on the caller's stream.  Both orders must give the same bits, repeatedly (no race between the parts),
    also for the warm-start pass structure, and the stage timers must cover the seven stages."""
    import torch
    import config5
    from paper_2205_03090_b200 import binding as B
    dev = torch.device("cuda:0")
    w = W.config3(200_000)
    z, P, T = (torch.from_numpy(a).to(dev) for a in (w.z, w.P, w.T))
    f = B.PTFlash.from_system(w.system)
    ref = {k: v.clone() for k, v in f.flash(z, P, T).items()}
    for rep in range(3):
        out = f.flash(z, P, T)
        for k in ("phase", "beta", "x", "y", "iters", "status"):
            assert torch.equal(out[k], ref[k]), k
    f.set_option("stage_profile", 1)
    out = f.flash(z, P, T)
    ms = f.stage_ms()
    assert len(ms) == 7 and all(m > 0 for m in ms)
    for k in ("phase", "beta", "x", "y", "iters", "status"):
        assert torch.equal(out[k], ref[k]), k
    st = f.stats()
    assert st["n_split"] >= st["n_probe_case3"] and st["n_two_phase"] == int((ref["phase"] == 2).sum())
    f.close()
    # warm start with skip-stability flags (two passes), forked vs single stream
    orc = oracle_mod.Oracle.from_system(W.system_co2_10())
    w5, lnK0, flags, info = config5.build(orc, 3000)
    g_fork = _gpu_flash(w5, 1, lnK0=lnK0, flags=flags)
    g_one = _gpu_flash(w5, 1, lnK0=lnK0, flags=flags, stage_profile=1)
    for k in ("phase", "beta", "x", "y", "iters", "status"):
        assert np.array_equal(g_fork[k], g_one[k]), k


@pytest.mark.gpu
@pytest.mark.parametrize("N", [1, 31, 33, 1025, 4133])
def test_outputs_stay_inside_their_buffers(N):
    """Guard words around every output array must survive a call (compute-sanitizer is not available on the GPU pool, so
    this is the bounds check for the stores of the user-visible arrays; cold call and warm-start call with flags)."""
    import torch
    from paper_2205_03090_b200 import binding as B
    dev = torch.device("cuda:0")
    w = W.config3(N)
    nc = w.system.nc
    z, P, T = (torch.from_numpy(a).to(dev) for a in (w.z, w.P, w.T))
    PAD, S64, S32 = 64, -7.25e300, -123456789

    def guarded(n_elem, dtype, sentinel):
        buf = torch.full((n_elem + 2 * PAD,), sentinel, dtype=dtype, device=dev)
        return buf, buf[PAD:PAD + n_elem]

    f = B.PTFlash.from_system(w.system)
    lnK_prev = None
    for warm in (False, True):
        bufs = {k: guarded(nc * N, torch.float64, S64) for k in ("x", "y", "lnK")}
        bufs.update({k: guarded(N, torch.float64, S64) for k in ("beta", "tpd")})
        bufs.update({k: guarded(N, torch.int32, S32) for k in ("phase", "iters", "status", "stab")})
        kw = {}
        if warm:
            kw = dict(lnK0=lnK_prev, flags=torch.ones(N, dtype=torch.uint8, device=dev))
        B.ptflash_flash_ex(f.h, N, z, P, T, bufs["beta"][1], bufs["x"][1], bufs["y"][1], bufs["phase"][1], bufs["iters"][1],
                           out_tpd_min=bufs["tpd"][1], out_lnK=bufs["lnK"][1], out_status=bufs["status"][1],
                           out_stab_iters=bufs["stab"][1], **kw)
        torch.cuda.synchronize()
        for k, (buf, view) in bufs.items():
            sent = S64 if buf.dtype == torch.float64 else S32
            assert bool((buf[:PAD] == sent).all()) and bool((buf[-PAD:] == sent).all()), (k, warm)
        assert bool(((bufs["phase"][1] == 1) | (bufs["phase"][1] == 2)).all())     # every element was written
        assert bool((bufs["beta"][1] != S64).all()) and bool((bufs["x"][1] != S64).all()) and bool((bufs["y"][1] != S64).all())
        lnK_prev = bufs["lnK"][1].clone()
    f.close()


def test_lnK0_flags_and_rejection(oracle_mod):
    """Warm-start sub-paths of ptflash_flash_ex (a14): flags 0..3 mixed in one call -- bit 1 (PTFLASH_FLAG_USE_LNK0: the
    caller's K seeds the probe and both stability starts, reading C19), bit 0 (skip stability), both -- plus rejected
    estimates (NaN, +-inf, |lnK0| > 700 -> Wilson, PTFLASH_ST_LNK0_REJECTED; the overflow failure of PAPER.md:363), plus
    skip-stability hints on mixtures that are in fact single phase (-> PTFLASH_ST_WARM_RESTART), all against the oracle."""
    N = 20000
    w = W.config3(N)
    orc = oracle_mod.Oracle.from_system(w.system)
    cold = orc.flash(w.z, w.P, w.T)
    two = cold["phase"] == 2
    n = np.arange(N)
    nc = w.system.nc
    wil = np.stack([orc.wilson(w.P[k], w.T[k]) for k in range(N)], axis=1)
    noise = np.stack([W.normal(909, n, 2 * i) for i in range(nc)])
    lnK0 = np.where(two[None, :], cold["lnK"] + 0.05 * noise, wil + 0.3 * noise)
    flags = np.minimum((W.uniform(909, n, 50) * 4).astype(np.uint8), 3)
    u = W.uniform(909, n, 51)
    comp = np.minimum((W.uniform(909, n, 52) * nc).astype(int), nc - 1)
    poison = {0: np.nan, 1: np.inf, 2: -np.inf, 3: 800.0, 4: -700.5}
    bad = np.zeros(N, dtype=bool)
    for k, v in poison.items():
        sel = (u >= 0.006 * k) & (u < 0.006 * (k + 1))
        lnK0[comp[sel], n[sel]] = v
        bad |= sel
    lnK0 = np.ascontiguousarray(lnK0)
    o = orc.flash(w.z, w.P, w.T, lnK0=lnK0, flags=flags)
    for engine in (1, 0):
        g = _gpu_flash(w, engine, lnK0=lnK0, flags=flags)
        g_cold = _gpu_flash(w, engine)
        # a skip-stability hint on a mixture the stability analysis calls stable is a contradiction the caller created:
        # whether the split from a noisy K still finds a (metastable) two-phase solution or fails and restarts depends on
        # the iteration path.  Such mixtures are compared unless the two sides ended with different restart flags.
        excuse = ((o["status"] ^ g["status"]) & 64) != 0
        assert excuse.sum() <= 5 and not np.any(excuse & two)
        check(w, g, o, excuse=excuse)
        rej_o, rej_g = (o["status"] & 32) != 0, (g["status"] & 32) != 0
        assert np.array_equal(rej_o, rej_g) and np.array_equal(rej_g, bad & (flags != 0))
        assert rej_g.sum() > 100
        # a rejected estimate means the plain Wilson path: bit-identical to the cold call
        for k in ("phase", "beta", "x", "y", "iters", "stab_iters"):
            assert np.array_equal(g[k][..., rej_g], g_cold[k][..., rej_g], equal_nan=True), k
        rs_g = (g["status"] & 64) != 0
        assert rs_g.sum() > 0.05 * N                                   # wrong hints on single-phase mixtures are dropped
        assert not np.any(rs_g & ((flags & 1) == 0))
        # bit 1 alone changes the stability starts (different iteration counts than the Wilson starts) but not the answer
        use = (flags == 2) & ~bad
        assert (g["stab_iters"][use] != g_cold["stab_iters"][use]).mean() > 0.02
        assert (np.abs(g["stab_iters"][use] - o["stab_iters"][use]) <= 2).mean() > 0.97    # the same starts as the oracle's
        assert np.array_equal(g["phase"][use], g_cold["phase"][use])
        # flags are ignored without lnK0, and lnK0 is ignored where flags == 0
        assert np.array_equal(g["beta"][flags == 0], g_cold["beta"][flags == 0])
        assert np.array_equal(_gpu_flash(w, engine, flags=flags)["beta"], g_cold["beta"])


def test_stats_match_oracle_counts(oracle_mod):
    """ptflash_get_stats (the paper's profiler columns, Table 4) against the same counts derived from the
    oracle's per-mixture outputs (probe case, per-stage iteration counts, status)."""
    import torch
    from paper_2205_03090_b200 import binding as B
    for cfg in (3, 2):
        N = 200_000
        w = W.CONFIGS[cfg](N)
        o = oracle_mod.Oracle.from_system(w.system).flash(w.z, w.P, w.T)
        g = _gpu_flash(w, 1)
        st = g["stats"]
        pc, stg = o["probe_case"], o["stage"]
        exp = dict(n_total=N, n_invalid=0, n_probe_case1=int((pc == 1).sum()), n_probe_case2=int((pc == 2).sum()),
                   n_probe_case3=int((pc == 3).sum()), n_stability=int(((pc == 1) | (pc == 2)).sum()),
                   n_stab_newton=int(stg[4].sum()), n_split=int(stg[7].sum()), n_split_newton=int(stg[8].sum()),
                   n_two_phase=int((o["phase"] == 2).sum()))
        print(cfg, {k: (st[k], v) for k, v in exp.items()})
        for k in ("n_total", "n_invalid", "n_stability", "n_two_phase", "n_split"):
            assert st[k] == exp[k], k
        # the three probe outcomes and the "needed the Newton stage" counts hinge on floating-point thresholds (theta in
        # (0,1), min < -1e-8, residual < 1e-10 after 9 iterations): equal up to a few borderline mixtures per million
        for k in ("n_probe_case1", "n_probe_case2", "n_probe_case3", "n_stab_newton", "n_split_newton"):
            assert abs(st[k] - exp[k]) <= max(2, 2e-5 * N), k
        assert np.array_equal(g["stab_iters"] > 0, stg[0] + stg[1] + stg[2] + stg[3] > 0)
        # iteration counts are path quantities (the CUDA stability Newton ends on a looser step criterion, C8), but close
        went = o["stab_iters"] > 0
        d = np.abs(g["stab_iters"] - o["stab_iters"])[went]
        print("stability iterations (both starts): |gpu - oracle| mean %.3f, <= 2 in %.4f of the mixtures" % (d.mean(), (d <= 2).mean()))
        assert (d <= 2).mean() > 0.97
        # the remaining columns of Table 4: per-start "went on to the trust-region stage", caps, max iterations per stage
        exp4 = dict(n_stab_tr=[int(stg[9].sum()), int(stg[10].sum())], n_stab_capped=[int(stg[11].sum()), int(stg[12].sum())],
                    n_split_capped=int(((o["status"] & 2) != 0).sum()), n_warm_restarts=0,
                    max_probe_iters=3, max_stab_ss_iters=[int(stg[0].max()), int(stg[1].max())],
                    max_stab_tr_iters=[int(stg[2].max()), int(stg[3].max())], max_split_ss_iters=int(stg[5].max()),
                    max_split_tr_iters=int(stg[6].max()))
        print(cfg, {k: (st[k], v) for k, v in exp4.items()})
        assert sum(st["n_stab_tr"]) == st["n_stab_newton"]
        for k in (0, 1):
            assert abs(st["n_stab_tr"][k] - exp4["n_stab_tr"][k]) <= max(2, 2e-5 * N)
            assert st["n_stab_capped"][k] == exp4["n_stab_capped"][k] == 0
            assert st["max_stab_ss_iters"][k] == exp4["max_stab_ss_iters"][k] == 9           # the SS cap of PAPER.md:79
            # trust-region iteration counts are path quantities (C8, C25): the maxima agree to a few iterations
            assert abs(st["max_stab_tr_iters"][k] - exp4["max_stab_tr_iters"][k]) <= 3
        assert st["n_split_capped"] == exp4["n_split_capped"] == 0 and st["n_warm_restarts"] == 0
        assert st["max_probe_iters"] == 3 and st["max_split_ss_iters"] == exp4["max_split_ss_iters"] == 9
        assert 1 <= st["max_split_tr_iters"] <= 60


def test_stability_only_mode(oracle_mod):
    """PTFLASH_OPT_STABILITY_ONLY: labels, tpd_min and K seeds without the phase split, against the oracle's
    stability-only mode; both engines; also through the caller's skip flag."""
    for cfg, N in ((3, 100_000), (4, 50_000), (1, 1000)):
        w = W.CONFIGS[cfg](N)
        orc = oracle_mod.Oracle.from_system(w.system)
        o = orc.flash(w.z, w.P, w.T, opts={"stability_only": 1})
        for engine in ((1, 0) if N <= 50_000 else (1,)):
            g = _gpu_flash(w, engine, stability_only=1)
            mism = np.nonzero(g["phase"] != o["phase"])[0]
            band = np.isfinite(o["tpd_min"]) & (o["tpd_min"] != 0) & (np.abs(o["tpd_min"]) < 1e-9)
            assert not len(np.setdiff1d(mism, np.nonzero(band)[0])), mism[:10]
            same = g["phase"] == o["phase"]
            un = same & (o["phase"] == 2)
            print(cfg, engine, "unstable", int(un.sum()), "stable", int((same & (o["phase"] == 1)).sum()))
            assert np.array_equal(g["x"], o["x"]) and np.array_equal(g["y"], o["y"])         # x = y = z, bit-exact
            assert np.all(np.isnan(g["beta"][g["phase"] == 2])) and np.array_equal(g["beta"][same & ~un], o["beta"][same & ~un])
            both = np.isfinite(o["tpd_min"]) & same
            assert np.abs(g["tpd_min"][both] - o["tpd_min"][both]).max() < 1e-9
            assert np.abs(g["lnK"][:, un] - o["lnK"][:, un]).max() < 1e-7                     # K seeds of the split
            assert np.all(g["lnK"][:, same & ~un] == 0.0) and np.all(g["iters"] <= 3)
            if engine == 1:
                st = g["stats"]
                assert st["n_two_phase"] == 0 and st["n_split_newton"] == 0 and st["n_split"] == int((g["phase"] == 2).sum())
        # the full flash labels the same mixtures "two-phase" except those whose split fails (status bit 8)
        gf = _gpu_flash(w, 1)
        gs = _gpu_flash(w, 1, stability_only=1)
        failed = (gf["status"] & 8) != 0
        assert np.array_equal(gf["phase"] == 2, (gs["phase"] == 2) & ~failed)
    # a skip-stability flag is a caller-side "unstable" verdict: reported as such, no work
    w = W.config3(3000)
    lnK0 = np.random.default_rng(5).normal(0, 1, w.z.shape)
    flags = (np.arange(w.N) % 3 == 0).astype(np.uint8)
    g = _gpu_flash(w, 1, lnK0=lnK0, flags=flags, stability_only=1)
    o = oracle_mod.Oracle.from_system(w.system).flash(w.z, w.P, w.T, lnK0=lnK0, flags=flags, opts={"stability_only": 1})
    assert np.array_equal(g["phase"], o["phase"]) and np.all(g["phase"][flags == 1] == 2)
    assert np.array_equal(g["lnK"][:, flags == 1], lnK0[:, flags == 1]) and np.all(np.isnan(g["tpd_min"][flags == 1]))


def test_derivative_output_and_batched_rachford_rice(oracle_mod):
    """NEXT-4: d beta / d K by the implicit-function formula (eq. 13) as a flash output and through the
    batched Rachford-Rice entry, against the oracle (which is pinned by finite differences of its own solver)."""
    import torch
    from paper_2205_03090_b200 import binding as B
    dev = torch.device("cuda:0")
    for cfg, N in ((3, 100_000), (2, 50_000), (1, 1000)):
        w = W.CONFIGS[cfg](N)
        orc = oracle_mod.Oracle.from_system(w.system)
        o = orc.flash(w.z, w.P, w.T)
        for engine in (1, 0):
            g = _gpu_flash(w, engine)
            two = (g["phase"] == 2) & (o["phase"] == 2)
            assert np.all(np.isnan(g["dbeta_dK"][:, g["phase"] != 2]))
            d_g, d_o = g["dbeta_dK"][:, two], o["dbeta_dK"][:, two]
            assert np.all(np.isfinite(d_g)) and np.all(d_g >= 0)
            # relative bar: the derivative inherits the 1e-8 absolute error of beta, x, y divided by sum (y - x)^2 / z
            rel = np.abs(d_g - d_o) / np.maximum(np.abs(d_o), 1e-6)
            print(cfg, engine, "two-phase", int(two.sum()), "max rel err of d beta / d K", rel.max())
            assert rel.max() < 1e-5 and np.median(rel) < 1e-9
        # the batched entry: perturbed K estimates (the initializer's use case), incl. rows without a window and bad input
        rng = np.random.default_rng(cfg)
        lnK = o["lnK"] + rng.normal(0, 0.3, o["lnK"].shape)
        lnK[:, o["phase"] != 2] = rng.normal(0, 1.0, (w.system.nc, int((o["phase"] != 2).sum())))
        lnK[:, 5] = 0.7            # no window
        lnK[0, 7] = np.nan         # invalid
        lnK[1, 9] = 800.0          # overflow guard
        ro = orc.rr_batch(np.where(np.isfinite(lnK) & (np.abs(lnK) <= 700), lnK, 0.0), w.z)
        ro["ok"][[7, 9]] = 0
        f = B.PTFlash.from_system(w.system)
        rg = {k: v.cpu().numpy() for k, v in f.rachford_rice(torch.from_numpy(lnK).to(dev), torch.from_numpy(w.z).to(dev)).items()}
        f.close()
        ok = ro["ok"] == 1
        assert np.array_equal(np.isfinite(rg["theta"]), ok) and not ok[5] and ok.mean() > 0.5
        assert np.all(np.isnan(rg["x"][:, ~ok])) and np.all(np.isnan(rg["dtheta_dK"][:, ~ok]))
        # theta is determined to ~ulp / |f'|: compare scaled by the window width (PAPER.md:525 stops at 1e-8 of it)
        K = np.exp(lnK[:, ok])
        width = np.minimum(1.0 / (1.0 - K.min(0)) - 1.0 / (1.0 - K.max(0)), 1.0)
        assert (np.abs(rg["theta"][ok] - ro["theta"][ok]) / width).max() < 1e-9
        assert np.abs(rg["x"][:, ok] - ro["x"][:, ok]).max() < 1e-8 and np.abs(rg["y"][:, ok] - ro["y"][:, ok]).max() < 1e-8
        rel = np.abs(rg["dtheta_dK"][:, ok] - ro["dtheta_dK"][:, ok]) / np.maximum(np.abs(ro["dtheta_dK"][:, ok]), 1e-9)
        print(cfg, "rr batch: solved", int(ok.sum()), "max rel err of d theta / d K", rel.max())
        assert rel.max() < 1e-6


@pytest.mark.parametrize("name,N", [("paper9", 100_000), ("paper4", 50_000), ("paper2", 50_000)])
def test_parity_paper_workloads(oracle_mod, name, N):
    """NEXT-3: the paper's own case studies (Tables 1-3; P in MPa), element by element against the oracle."""
    w = W.CONFIGS[name](N)
    o = oracle_mod.Oracle.from_system(w.system).flash(w.z, w.P, w.T)
    # engine 1 only at these sizes: engine 0 follows the oracle's statement order, so agreeing with it is
    # not independent evidence; it stays in the small parity tests
    for engine in (1,):
        g = _gpu_flash(w, engine)
        rep = compare(w, g, o)
        rows = adjudicate(oracle_mod, w, g, o, rep["bad"])
        for r in rows:
            print("  adjudicated:", r)
        print(name, engine, {k: v for k, v in rep.items() if k not in ("messages", "bad", "band")})
        assert rep["n_hard"] == 0, "\n".join(rep["messages"])
        assert all(r["attributed"] != "BUG" for r in rows) and len(rows) <= max(1, N // 50_000)
        assert rep["max_err_single"] == 0.0 and rep["beta_convention_mismatch"] == 0
    st = g["stats"] if False else _gpu_flash(w, 1)["stats"]
    print(name, "two-phase share %.4f (paper, 9 components: 0.4134), probe-proved share %.4f (paper: 0.3744)"
          % (st["n_two_phase"] / N, st["n_probe_case3"] / N))


def test_pipelined_host_call(oracle_mod):
    """ptflash_flash_host_async / ptflash_host_wait: several batches in flight (different inputs, one output set per batch)
    give bit-identical results to the device-buffer call, also when a slot is reused; sync host call alike (chunked)."""
    import torch
    from paper_2205_03090_b200 import binding as B
    N = 150_000
    f = B.PTFlash.from_system(W.system_co2_10())
    batches = [W.config3(N, offset=k * N) for k in range(5)]
    ref = [_gpu_flash(w, 1) for w in batches]
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
    hin = [(pin(w.z), pin(w.P), pin(w.T)) for w in batches]
    hout = [dict(beta=torch.empty(N, dtype=torch.float64).pin_memory(), x=torch.empty(10, N, dtype=torch.float64).pin_memory(),
                 y=torch.empty(10, N, dtype=torch.float64).pin_memory(), phase=torch.empty(N, dtype=torch.int32).pin_memory(),
                 iters=torch.empty(N, dtype=torch.int32).pin_memory()) for _ in batches]
    for (z, P, T), o in zip(hin, hout):
        B.ptflash_flash_host_async(f.h, N, z, P, T, o["beta"], o["x"], o["y"], o["phase"], o["iters"])
    B.ptflash_host_wait(f.h)
    for k, (o, r) in enumerate(zip(hout, ref)):
        for key in ("beta", "x", "y", "phase", "iters"):
            assert np.array_equal(o[key].numpy(), r[key], equal_nan=True), (k, key)
    assert f.stats()["n_two_phase"] == int((ref[-1]["phase"] == 2).sum())
    # the chunked synchronous call (4 chunks of 37,500 here) on the same handle
    o = hout[0]
    for key in o:
        o[key].zero_()
    z, P, T = hin[3]
    B.ptflash_flash_host(f.h, N, z, P, T, o["beta"], o["x"], o["y"], o["phase"], o["iters"])
    for key in ("beta", "x", "y", "phase", "iters"):
        assert np.array_equal(o[key].numpy(), ref[3][key], equal_nan=True), key
    st = f.stats()
    assert st["n_total"] == N and st["n_two_phase"] == int((ref[3]["phase"] == 2).sum())
    f.close()


def test_host_call_row_by_row_copies():
    """ptflash_flash_host moves its strided SoA slices with 2D copies, whose pitch is limited to 2^31 - 1 bytes: from
    N = 2^28 mixtures on it falls back to one copy per component row.  That size does not fit a test; the
    host_row_copies option takes the same path at an ordinary size.  Both must give the bits of the device-buffer call,
    also on a chunk boundary that is not a multiple of anything (2 chunks here)."""
    import torch
    from paper_2205_03090_b200 import binding as B
    N = 70_001
    w = W.config3(N, offset=123_456)
    ref = _gpu_flash(w, 1)
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
    z, P, T = pin(w.z), pin(w.P), pin(w.T)
    for rows in (1, 0):
        f = B.PTFlash.from_system(w.system, host_row_copies=rows)
        assert B.ptflash_get_option(f.h, "host_row_copies") == rows
        o = dict(beta=torch.full((N,), -7.0, dtype=torch.float64).pin_memory(), x=torch.full((10, N), -7.0, dtype=torch.float64).pin_memory(),
                 y=torch.full((10, N), -7.0, dtype=torch.float64).pin_memory(), phase=torch.full((N,), -7, dtype=torch.int32).pin_memory(),
                 iters=torch.full((N,), -7, dtype=torch.int32).pin_memory())
        B.ptflash_flash_host(f.h, N, z, P, T, o["beta"], o["x"], o["y"], o["phase"], o["iters"])
        for key in ("beta", "x", "y", "phase", "iters"):
            assert np.array_equal(o[key].numpy(), ref[key], equal_nan=True), (rows, key)
        assert f.stats()["n_two_phase"] == int((ref["phase"] == 2).sum())
        f.close()
    with pytest.raises(B.PTFlashError):
        B.PTFlash.from_system(w.system, host_row_copies=2)


def test_rachford_rice_leaves_the_flash_statistics_alone():
    """ptflash_rachford_rice on another stream must not change what ptflash_get_stats waits for and reports:
    the counters belong to the last flash and to the stream that flash ran on."""
    import torch
    from paper_2205_03090_b200 import binding as B
    dev = torch.device("cuda:0")
    w = W.config3(200_000)
    f = B.PTFlash.from_system(w.system)
    z, P, T = (torch.from_numpy(a).to(dev) for a in (w.z, w.P, w.T))
    lnK = torch.zeros_like(z)
    lnK[0] = 1.0
    lnK[1] = -1.0
    s_flash, s_rr = torch.cuda.Stream(), torch.cuda.Stream()
    with torch.cuda.stream(s_flash):
        out = f.flash(z, P, T)
    s_flash.synchronize()
    want = f.stats()
    with torch.cuda.stream(s_flash):
        out = f.flash(z, P, T)                      # still running when the Rachford-Rice call below is made ...
    with torch.cuda.stream(s_rr):
        rr = f.rachford_rice(lnK, z)                # ... on a stream that finishes long before it
    got = f.stats()                                 # has to wait for the flash, not for the Rachford-Rice stream
    assert got == want and got["n_total"] == w.N and got["n_two_phase"] == int((out["phase"] == 2).sum())
    torch.cuda.synchronize()
    assert torch.isfinite(rr["theta"]).all()
    f.close()


def test_second_device_keeps_current_device():
    """A handle created on cuda:1 is used and destroyed while cuda:0 is current: the caller's device is
    restored by every entry point and the results equal those of cuda:0."""
    import torch
    from paper_2205_03090_b200 import binding as B
    if torch.cuda.device_count() < 2:
        pytest.skip("needs two GPUs")
    w = W.config3(5000)
    ref = _gpu_flash(w, 1)
    torch.cuda.set_device(1)
    f = B.PTFlash.from_system(w.system)
    torch.cuda.set_device(0)
    d1 = torch.device("cuda:1")
    z, P, T = (torch.from_numpy(a).to(d1) for a in (w.z, w.P, w.T))
    with torch.cuda.device(1):
        st = torch.cuda.current_stream().cuda_stream
    out = f.flash(z, P, T, stream=st)
    assert torch.cuda.current_device() == 0
    f.stats()
    assert torch.cuda.current_device() == 0
    for k in ("phase", "beta", "x", "y"):
        assert np.array_equal(out[k].cpu().numpy(), ref[k], equal_nan=True), k
    f.close()
    assert torch.cuda.current_device() == 0


@pytest.mark.parametrize("nproc", [1, 2])
def test_bench_under_torchrun(nproc, tmp_path):
    """bench.py launched the way the driver launches it for N > 1 (its NCCL init, per-rank shard offsets and
    max-over-ranks timing had never run anywhere).  With one process the same code path runs on a 1-GPU box (the group is
    created whenever torchrun set one up); with two it needs two GPUs.  Rank 0 prints ONE JSON line; the job-wide value
    is ranks x N x steps / max-over-ranks time, so two ranks on two GPUs must land near twice the one-rank figure."""
    import json, subprocess, sys, torch
    if torch.cuda.device_count() < nproc:
        pytest.skip(f"needs {nproc} GPUs")
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    n = 200_000
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={nproc}", "--master-addr", "127.0.0.1",
           "--master-port", str(29500 + 17 * nproc + os.getpid() % 400), os.path.join(root, "bench.py"), "--gpus", str(nproc),
           "--steps", "3", "--warmup", "3", "--no-cpu-baseline", "--mixtures", str(n)]
    r = subprocess.run(cmd, capture_output=True, text=True, cwd=root, timeout=600)
    assert r.returncode == 0, r.stderr[-3000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1, r.stdout[-2000:]                      # rank 0 alone prints
    d = json.loads(lines[0])
    assert d["n_gpus"] == nproc and d["steps"] == 3 and d["scaling"] == "weak" and d["config"]["mixtures_per_step"] == n
    assert d["gpu_launches"] > 0 and d["roofline"]["frac"] > 0.05 and d["e2e"]["value"] > 0
    # whole-job throughput: ranks x n mixtures per step over the slowest rank's time
    assert abs(d["value"] - nproc * n / (d["ms_per_step"] * 1e-3)) < 1e-6 * d["value"]
    print(f"torchrun x{nproc}: {d['value'] / 1e6:.1f} M flashes/s, {d['ms_per_step']:.3f} ms per step of {n} mixtures per rank")


def _ulps(y, ref):
    """|y - ref| in units of the spacing of doubles at ref (ref: numpy longdouble)."""
    r64 = ref.astype(np.float64)
    return np.abs((y.astype(np.longdouble) - ref) / np.spacing(np.abs(r64)).astype(np.longdouble)).astype(np.float64)


def test_math_routines_against_libm():
    """The lean exp / log / reciprocal routines of csrc/ptflash_math.cuh through ptflash_math_probe against libm in
    extended precision: <= 2 ulp on the stated ranges, and the documented behaviour at the clamps."""
    import torch
    from paper_2205_03090_b200 import binding as B
    dev = torch.device("cuda:0")
    rng = np.random.default_rng(20220503)
    M = 400_000
    L = np.longdouble

    def run(fn, x):
        xd = torch.from_numpy(np.ascontiguousarray(x, dtype=np.float64)).to(dev)
        yd = torch.empty_like(xd)
        B.ptflash_math_probe(fn, xd.numel(), xd, yd)
        torch.cuda.synchronize()
        return yd.cpu().numpy()

    lognormal = np.exp(rng.uniform(-700.0, 700.0, M))
    cases = {
        "exp_fast": (np.concatenate([rng.uniform(-708.0, 709.0, M), rng.uniform(-1e-3, 1e-3, 1000), [0.0, -708.0, 709.0, 1e-300]]),
                     lambda x: np.exp(x.astype(L))),
        "exp_tab": (np.concatenate([rng.uniform(-700.0, 709.0, M), rng.uniform(-1e-3, 1e-3, 1000), [0.0, -700.0, 709.0]]),
                    lambda x: np.exp(x.astype(L))),
        "log_fast": (np.concatenate([lognormal, rng.uniform(0.5, 2.0, M), [1.0, np.sqrt(2.0), np.nextafter(np.sqrt(2.0), 2), 2.2250738585072014e-308, 1.7e308]]),
                     lambda x: np.log(x.astype(L))),
        "log1p_fast": (np.concatenate([rng.uniform(0.0, 1.0, M), np.exp(rng.uniform(-40, 0, M)) * 0.999, [0.0, 0.41421356237309503, 0.4142135623730951, 0.9999999999999999]]),
                       lambda x: np.log1p(x.astype(L))),
        "rcp_fast": (np.concatenate([np.exp(rng.uniform(-300, 300, M)) * rng.choice([-1.0, 1.0], M), [1.0, -1.0, 3.0]]),
                     lambda x: L(1) / x.astype(L)),
        "div_fast_1": (np.exp(rng.uniform(-300, 300, M)), lambda x: L(1) / x.astype(L)),
        "rsqrt_fast": (np.exp(rng.uniform(-600, 600, M)), lambda x: L(1) / np.sqrt(x.astype(L))),
        "sqrt_fast": (np.concatenate([np.exp(rng.uniform(-600, 600, M)), [0.0, 1.0, 4.0]]), lambda x: np.sqrt(x.astype(L))),
    }
    # exp_tab: table value (0.5 ulp) x degree-5 polynomial x product rounding; log: reciprocal + series + two-term ln 2 sum
    bound = {"exp_tab": 2.5, "log_fast": 2.5, "log1p_fast": 2.5, "exp_fast": 1.0, "rcp_fast": 1.0, "div_fast_1": 1.0, "rsqrt_fast": 1.0, "sqrt_fast": 1.0}
    worst = {}
    for fn, (x, ref) in cases.items():
        y = run(fn, x)
        r = ref(x)
        ok = r != 0
        u = np.zeros(len(x))
        u[ok] = _ulps(y[ok], r[ok])
        assert np.all(np.isfinite(y)), fn
        assert np.all(y[~ok] == 0.0), fn
        print(f"{fn}: max {u.max():.3f} ulp, mean {u.mean():.3f} ulp over {len(x)} arguments")
        worst[fn] = (float(u.max()), float(x[np.argmax(u)]))
    for fn, (u, x) in worst.items():
        assert u <= bound.get(fn, 2.0), (fn, u, x)
    # ~2^-40 reciprocal used inside self-correcting iterations
    x = np.exp(rng.uniform(-300, 300, M))
    assert np.abs(run("rcp_nr1", x) * x - 1.0).max() < 2.0 ** -38
    # clamps: exp_fast below -708 and exp_tab below -700 return the value at the clamp (finite, normal), never 0 or NaN
    lo = np.array([-708.0, -709.0, -745.0, -1000.0, -1e300])
    assert np.all(run("exp_fast", lo) == run("exp_fast", np.full(5, -708.0)))
    lo = np.array([-700.0, -701.0, -745.0, -1000.0, -1e300])
    assert np.all(run("exp_tab", lo) == run("exp_tab", np.full(5, -700.0)))
    assert np.all(run("exp_tab", lo) > 2.2250738585072014e-308)
    # sqrt_fast(0) = 0 exactly; rcp_fast(0) is documented as NaN (the kernels never divide by an exact zero)
    assert run("sqrt_fast", np.zeros(3)).tolist() == [0.0, 0.0, 0.0]
    assert np.all(np.isnan(run("rcp_fast", np.zeros(3))))


MAX_ATTRIBUTED_MISSES = 3    # per 10^6 mixtures (configs 2-4): two-phase mixtures above 1e-8, each attributed (see adjudicate)
MAX_ADJUDICATED_GAP = 1e-6   # ... and none of them further than this from the oracle, whatever the attribution
ISOFUGACITY_TOL = 2e-9       # max_i |ln f_i^L - ln f_i^V| of a two-phase CUDA result, recomputed in numpy (measured: <= 4.1e-10 over every full-size batch, config 5 included; 1e-9 is asserted of the oracle)


def _full_size(oracle_mod, w, g, o, lnK0=None, flags=None, max_misses=MAX_ATTRIBUTED_MISSES, excuse=None, max_gap=MAX_ADJUDICATED_GAP):
    """Invariants on every mixture + element-by-element oracle parity on every mixture (the oracle flashes ~1e6
    mixtures per second on the box's host cores).  Misses above 1e-8 are adjudicated, listed and bounded."""
    N = w.N
    assert set(np.unique(g["phase"])) <= {1, 2}
    two = g["phase"] == 2
    b = g["beta"]
    assert np.all((b[two] > 0) & (b[two] < 1)) and np.all(np.isin(b[~two], (0.0, 1.0)))
    assert np.abs(w.z - b * g["y"] - (1 - b) * g["x"])[:, two].max() < 1e-10          # (1a)
    # (1b); worst case is a Newton finish with beta within 1e-5 of 0 or 1 (x = (z - nV)/(1 - beta))
    assert np.abs(g["x"].sum(0) - 1).max() < 1e-9 and np.abs(g["y"].sum(0) - 1).max() < 1e-9
    assert (g["status"] & 3).sum() == 0                                                   # no iteration cap hit
    # (2) iso-fugacity and the stability verdict on the CUDA results by themselves: ln phi recomputed here in numpy
    # (tests/srk_check.py, pinned against the oracle on the CPU) -- a check that does not pass through the oracle's
    # iteration, tolerances or acceptance rules, which were tuned side by side with the kernels
    import srk_check
    idx2 = np.nonzero(two)[0]
    res = np.concatenate([srk_check.isofugacity_residual(w.system, w.P[c], w.T[c], g["x"][:, c], g["y"][:, c])
                          for c in np.array_split(idx2, max(1, len(idx2) // 200_000))])
    worst = idx2[np.argsort(res)[-3:]]
    print(f"  iso-fugacity residual max_i |ln f_i^L - ln f_i^V| of the {len(idx2)} two-phase CUDA results: max {res.max():.3e}, "
          f"99.99 % below {np.quantile(res, 0.9999):.3e}; worst n = {worst.tolist()}")
    assert res.max() < ISOFUGACITY_TOL, f"iso-fugacity violated at n = {worst.tolist()}: {np.sort(res)[-3:]}"
    # a mixture reported single phase has no trial phase with a TPD below the band -- unless the split of an unstable feed
    # failed and says so (PTFLASH_ST_SPLIT_FAILED); NaN = stability analysis skipped on the caller's word
    tpd1 = g["tpd_min"][~two & ((g["status"] & 8) == 0)]
    assert np.all(np.isnan(tpd1) | (tpd1 >= -1e-9))
    rep = compare(w, g, o, excuse=excuse)
    print({k: v for k, v in rep.items() if k not in ("messages", "bad", "band")})
    for n in rep["band"]:
        print(f"  in-band label mismatch n={n}: tpd_min oracle {o['tpd_min'][n]:.3e} gpu {g['tpd_min'][n]:.3e}")
    assert rep["n_hard"] == 0, "\n".join(rep["messages"])
    assert rep["in_band"] <= max(1, int(np.ceil(MAX_BAND_PER_MILLION * N / 1e6)))
    assert rep["max_err_single"] == 0.0 and rep["beta_convention_mismatch"] == 0
    rows = adjudicate(oracle_mod, w, g, o, rep["bad"], lnK0, flags)
    for r in rows:
        print("  miss above 1e-8:", r)
    assert all(r["attributed"] != "BUG" for r in rows), "a miss above 1e-8 that neither the oracle's rounding nor conditioning explains"
    assert len(rows) <= max_misses
    # whatever the attribution, an adjudicated miss stays small in absolute terms.  Not so on config 5, whose
    # mixtures all sit within 5 % of their phase boundary: there a handful per 1e6 are so ill-conditioned that the double
    # oracle, the long-double oracle and the CUDA path disagree in the first digits of beta (VERDICT r2, weak point 4: they
    # need a status bit of their own, which does not exist yet) -- that caller passes max_gap=None and lists them.
    if max_gap is not None:
        assert all(r["gap_gpu_oracle"] <= max_gap for r in rows), [r for r in rows if r["gap_gpu_oracle"] > max_gap]
    rep["misses"] = rows
    return rep


@pytest.mark.parametrize("cfg,N", [(2, 1_000_000), (3, 1_000_000), (4, 1 << 16), (4, 1 << 20), (4, 1 << 22), (4, 1 << 24)])
def test_full_size_parity(oracle_mod, cfg, N):
    """BASELINE sizes (configs[1..3], the scaling sweep of configs[3] from 2^16 to 2^24; config 3 at 1e6 is the launch
    configuration bench.py times; at these sizes the persistent Newton kernels refill their lanes ~40 times and more):
    EVERY mixture against the oracle."""
    w = W.CONFIGS[cfg](N)
    g = _gpu_flash(w, 1)
    o = oracle_mod.Oracle.from_system(w.system).flash(w.z, w.P, w.T)
    # attributed misses above 1e-8 (near-critical mixtures, each adjudicated against the long double oracle): at most
    # MAX_ATTRIBUTED_MISSES per call up to 2^22 mixtures, and 1 per 2^22 above
    rep = _full_size(oracle_mod, w, g, o, max_misses=max(MAX_ATTRIBUTED_MISSES, N >> 22))
    assert 0.10 < rep["two_phase"] / N < 0.35
    assert (g["iters"] == o["iters"]).mean() > 0.98


def test_full_size_config5_warm_and_cold(oracle_mod):
    """BASELINE configs[4] at its stated size (1e6 mixtures within 5 % of their phase boundary; PTFLASH_TEST_CONFIG5_N
    overrides): warm (caller lnK0 + skip-stability flags) and cold calls, every mixture against the oracle."""
    import config5
    N = int(os.environ.get("PTFLASH_TEST_CONFIG5_N", "1000000"))
    orc = oracle_mod.Oracle.from_system(W.system_co2_10())
    w, lnK0, flags, info = config5.build_cached(orc, N)
    o_cold = info["cold"]
    o_warm = orc.flash(w.z, w.P, w.T, lnK0=lnK0, flags=flags)
    g_cold = _gpu_flash(w, 1)
    # every mixture of this workload is within 5 % of its phase boundary, where G is flat: more conditioning-limited misses
    # than in configs 2-4 (each one adjudicated against the long double oracle and listed)
    rc = _full_size(oracle_mod, w, g_cold, o_cold, max_misses=max(3, int(20e-6 * N)), max_gap=None)
    o_restarted = (o_warm["status"] & 64) != 0
    # Which hints fail is a property of the iteration path next to the boundary.  With PTFLASH_OPT_HINT_ETA_SEARCH = 1 the
    # hinted splits take the oracle's restricted step (eta search of B.4a) and the restart sets agree up to borderline
    # cases; the default takes the truncated modified-Cholesky step of C25: same answers, but a bounded, reported share of
    # the hints fails or survives differently.  A mixture restarted on one side only is compared after the restart all the
    # same (the cold answer); it is left out only if the LABELS differ, i.e. the hinted split found two phases on one side
    # where the cold stability analysis (the other side) says single phase.
    for eta, bound in ((1, max(3, 1e-5 * N)), (0, max(3, 4e-3 * N))):
        g_warm = _gpu_flash(w, 1, lnK0=lnK0, flags=flags, hint_eta_search=eta)
        restarted = (g_warm["status"] & 64) != 0
        differ = restarted != o_restarted
        print("config5 warm, hint_eta_search = %d: restarts gpu %d oracle %d, on one side only %d" % (eta, restarted.sum(), o_restarted.sum(), differ.sum()))
        assert differ.sum() <= bound
        excuse = differ & (g_warm["phase"] != o_warm["phase"])
        assert excuse.sum() <= max(1, 2e-5 * N)
        rw = _full_size(oracle_mod, w, g_warm, o_warm, lnK0, flags, max_misses=max(3, int(20e-6 * N)), excuse=excuse, max_gap=None)
    assert 0.4 < rc["two_phase"] / N < 0.6
    two = (g_warm["phase"] == 2) & (g_cold["phase"] == 2)
    print("config5 N=%d: two-phase %.3f, restarts gpu %d oracle %d; mean iters (two-phase) warm %.2f cold %.2f" %
          (N, rc["two_phase"] / N, restarted.sum(), o_restarted.sum(), g_warm["iters"][two].mean(), g_cold["iters"][two].mean()))
