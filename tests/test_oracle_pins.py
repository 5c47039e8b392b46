"""Pins for the CPU oracle (oracle/ptflash_oracle.cpp): each test checks the oracle against something
the paper or the mathematics fixes, NOT against itself -- closed forms, invariants, textbook special
cases, brute force on tiny inputs.  A plausible mistake (dropped term, wrong sign/index, transposed
operand) fails at least one of them.  Citations are PAPER.md:<line>.  All CPU, -m "not gpu".
"""
import sys
from pathlib import Path

import numpy as np
import pytest

from paper_2205_03090_b200 import workloads as W

RNG = np.random.default_rng(20220503)


@pytest.fixture(scope="module")
def sys10(oracle_mod):
    return oracle_mod.Oracle.from_system(W.system_co2_10())


@pytest.fixture(scope="module")
def sys2(oracle_mod):
    return oracle_mod.Oracle.from_system(W.system_binary())


# ------------------------------------------------------------------------------------------------
# input generator (shared module): SplitMix64 test vectors, ranges, simplex
# ------------------------------------------------------------------------------------------------
def test_splitmix64_vectors():
    # published SplitMix64 sequence for seed 0: outputs are mix64(k * golden), k = 1, 2, 3
    g = 0x9E3779B97F4A7C15
    got = W.mix64(np.array([g, (2 * g) % 2**64, (3 * g) % 2**64], dtype=np.uint64))
    assert [int(v) for v in got] == [0xE220A8397B1DCDAF, 0x6E789E6AA1B965F4, 0x06C45D188009454F]


def test_workload_shapes_and_ranges():
    for cfg, (Tlo, Thi, Plo, Phi) in {1: (250, 550, 1, 150), 2: (200, 600, 1, 200), 3: (220, 500, 5, 300),
                                       4: (220, 500, 5, 300)}.items():
        w = W.CONFIGS[cfg](5000)
        assert w.z.shape == (w.system.nc, 5000)
        assert np.all((w.T > Tlo) & (w.T < Thi)) and np.all((w.P > Plo) & (w.P < Phi))
        assert np.all(w.z > 0) and np.allclose(w.z.sum(0), 1.0, atol=1e-14)
        # prefix property of the counter-based generator
        w2 = W.CONFIGS[cfg](100, offset=200)
        assert np.array_equal(w2.P, w.P[200:300]) and np.array_equal(w2.z, w.z[:, 200:300])
    w3 = W.config3(20000)
    assert abs(w3.z[8].mean() - (0.4 + 0.06)) < 5e-3          # 0.6 * 1/10 + 0.4
    w4 = W.config4(20000)
    assert abs(w4.z.mean() - 0.1) < 1e-12 and abs(w4.z.var() - 0.1 * 0.9 / 6.0) < 2e-3   # Dirichlet(1/2): var = m(1-m)/(a0+1)


# ------------------------------------------------------------------------------------------------
# O1 setup: A.2d-g PAPER.md:420-427
# ------------------------------------------------------------------------------------------------
def test_setup_constants(sys10):
    s = W.system_co2_10()
    P, T = 57.3, 333.3
    Ai, Bi, Aij = sys10.setup(P, T)
    m = 0.480 + 1.574 * s.omega - 0.176 * s.omega**2
    Tr = T / s.Tc
    alpha = (1 + m * (1 - np.sqrt(Tr))) ** 2
    # ratio A_i/B_i = (0.42748/0.08664) alpha_i / Tr_i  (R cancels)
    np.testing.assert_allclose(Ai / Bi, 0.42748 / 0.08664 * alpha / Tr, rtol=1e-13)
    np.testing.assert_allclose(Bi, 0.08664 * (P / s.Pc) / Tr, rtol=1e-14)
    # mixing rule A.2b with the config-3 BIPs; symmetric
    np.testing.assert_allclose(Aij, (1 - s.kij) * np.sqrt(np.outer(Ai, Ai)), rtol=1e-13)
    assert Aij[0, 8] == pytest.approx(0.88 * np.sqrt(Ai[0] * Ai[8]), rel=1e-13)
    assert Aij[8, 9] == pytest.approx(1.02 * np.sqrt(Ai[8] * Ai[9]), rel=1e-13)
    # alpha = 1 at T = Tc: pure component at its critical point has A = 0.42748, B = 0.08664
    for i in (0, 8):
        Ai_c, Bi_c, _ = sys10.setup(s.Pc[i], s.Tc[i])
        assert Ai_c[i] == pytest.approx(0.42748, rel=1e-14) and Bi_c[i] == pytest.approx(0.08664, rel=1e-14)


def test_critical_point_cubic_coefficients():
    # SRK critical point: rho1 ~ 1/3, rho0 ~ 1/27 (triple root Z = 1/3) with the rounded literals
    A, B = 0.42748, 0.08664
    assert A - B * (1 + B) == pytest.approx(1 / 3, abs=3e-7)
    assert A * B == pytest.approx(1 / 27, abs=3e-7)


# ------------------------------------------------------------------------------------------------
# cubic A.3-A.5 PAPER.md:431-445
# ------------------------------------------------------------------------------------------------
def _rand_AB(n):
    A = 10 ** RNG.uniform(-4, np.log10(20), n)
    B = 10 ** RNG.uniform(-5, np.log10(0.9), n)
    return A, B


def test_cubic_vieta_and_closed_form(sys2):
    A, B = _rand_AB(4000)
    n3 = 0
    for a, b in zip(A, B):
        r = sys2.cubic_roots(a, b)
        rho0, rho1 = a * b, a - b * (1 + b)
        f = lambda Z: ((Z - 1) * Z + rho1) * Z - rho0
        df = lambda Z: (3 * Z - 2) * Z + rho1
        scale = max(1.0, abs(rho1), abs(rho0))
        for Z in r:
            # residual small against the local conditioning |f'| * ulp
            assert abs(f(Z)) <= 64 * np.finfo(float).eps * scale * max(1.0, abs(Z)) ** 3
        rc = sys2.cubic_roots(a, b, closed=True)
        if len(r) == 3 and len(rc) == 3:
            n3 += 1
            # Vieta: sum = 1, sum of pairs = rho1, product = rho0
            assert r.sum() == pytest.approx(1.0, abs=1e-12)
            assert r[0] * r[1] + r[0] * r[2] + r[1] * r[2] == pytest.approx(rho1, abs=1e-12 * scale)
            assert r.prod() == pytest.approx(rho0, abs=1e-12 * scale)
            # closed form after a Newton polish of its roots
            rc = np.array([Z - f(Z) / df(Z) if df(Z) != 0 else Z for Z in rc])
            sep = min(r[1] - r[0], r[2] - r[1])
            if sep > 1e-4:
                np.testing.assert_allclose(r, rc, rtol=0, atol=1e-9)
        elif len(r) == 1 and len(rc) == 1:
            assert r[0] == pytest.approx(rc[0], rel=1e-6)
    assert n3 > 200  # the three-root branch was exercised


def test_cubic_fixed_values():
    # f(B) = -2B^2 and f(1+B) = A for every A, B (used to choose the Newton side, C15)
    for a, b in zip(*_rand_AB(50)):
        rho0, rho1 = a * b, a - b * (1 + b)
        f = lambda Z: Z**3 - Z**2 + rho1 * Z - rho0
        assert f(b) == pytest.approx(-2 * b * b, abs=1e-12 * max(1, a))
        assert f(1 + b) == pytest.approx(a, rel=1e-10)


def test_root_choice_admissible_and_min_gibbs(sys2):
    # SURVEY probe case: A=0.01, B=0.5 has roots -0.490, -0.0068, 1.497 -> only the last is admissible (C3)
    r = sys2.cubic_roots(0.01, 0.5)
    assert len(r) == 3 and r[0] < 0 and r[1] < 0.5
    assert sys2.choose_root(0.01, 0.5) == pytest.approx(r[2], rel=1e-15)
    # three admissible roots: choice is the smaller g of the two outer roots (C4)
    cnt = 0
    for a, b in zip(*_rand_AB(3000)):
        r = sys2.cubic_roots(a, b)
        adm = r[r > b]
        Z = sys2.choose_root(a, b)
        assert Z > b
        if len(adm) >= 2:
            cnt += 1
            g = lambda z: z - 1 - np.log(z - b) - a / b * np.log(1 + b / z)
            best = adm[0] if g(adm[0]) <= g(adm[-1]) else adm[-1]
            assert Z == pytest.approx(best, rel=1e-14)
            assert not np.isclose(Z, adm[1] if len(adm) == 3 else -1, rtol=1e-9)  # never the middle root
    assert cnt > 50


def test_ideal_gas_limit(sys10):
    z = np.full(10, 0.1)
    lp, Z = sys10.lnphi(1e-6, 400.0, z)
    assert Z == pytest.approx(1.0, abs=1e-6) and np.abs(lp).max() < 1e-6


# ------------------------------------------------------------------------------------------------
# lnphi A.6 PAPER.md:447-450 and its composition derivative (formula derived in DESIGN.md)
# ------------------------------------------------------------------------------------------------
def _rand_comp(nc):
    c = RNG.exponential(size=nc)
    return c / c.sum()


def test_lnphi_sum_rule(sys10):
    # sum c_i lnphi_i = g(Z) = Z - 1 - ln(Z-B) - (A/B) ln(1+B/Z): ties A.6 to the residual Gibbs energy (C4)
    for _ in range(200):
        P, T, c = RNG.uniform(5, 300), RNG.uniform(220, 500), _rand_comp(10)
        Ai, Bi, Aij = sys10.setup(P, T)
        A, B = c @ Aij @ c, c @ Bi
        lp, Z = sys10.lnphi(P, T, c)
        g = Z - 1 - np.log(Z - B) - A / B * np.log(1 + B / Z)
        assert c @ lp == pytest.approx(g, abs=1e-12)
        assert abs(Z**3 - Z**2 + (A - B - B * B) * Z - A * B) < 1e-13 * max(1, A)


def test_lnphi_matches_textbook_form(sys10):
    # A.6 exactly as printed (b_i/b, (a alpha)_ij, A/B) evaluated with numpy from the setup arrays
    for _ in range(100):
        P, T, c = RNG.uniform(5, 300), RNG.uniform(220, 500), _rand_comp(10)
        Ai, Bi, Aij = sys10.setup(P, T)
        A, B = c @ Aij @ c, c @ Bi
        lp, Z = sys10.lnphi(P, T, c)
        ref = Bi / B * (Z - 1) - np.log(Z - B) + A / B * (Bi / B - 2.0 / A * (Aij @ c)) * np.log(1 + B / Z)
        np.testing.assert_allclose(lp, ref, rtol=0, atol=1e-12)


def test_dlnphi_finite_difference_symmetry_gibbs_duhem(sys10):
    for _ in range(40):
        P, T, c = RNG.uniform(5, 300), RNG.uniform(220, 500), _rand_comp(10)
        lp, Z, M = sys10.lnphi(P, T, c, deriv=True)
        np.testing.assert_allclose(M, M.T, atol=1e-12 * max(1, np.abs(M).max()))        # symmetry
        np.testing.assert_allclose(c @ M, 0, atol=1e-11 * max(1, np.abs(M).max()))       # Gibbs-Duhem
        h = 1e-6
        for j in (0, 3, 8, 9):
            n1, n2 = c.copy(), c.copy()
            n1[j] += h
            n2[j] -= h
            l1, Z1 = sys10.lnphi(P, T, n1 / n1.sum())
            l2, Z2 = sys10.lnphi(P, T, n2 / n2.sum())
            if abs(Z1 - Z2) > 1e-3:   # root switch between the two FD points
                continue
            np.testing.assert_allclose(M[:, j], (l1 - l2) / (2 * h), atol=2e-7 * max(1, np.abs(M).max()))


def test_pure_component_saturation_matches_acentric_factor_definition(oracle_mod):
    # omega := -log10(Psat/Pc at Tr = 0.7) - 1.  Soave fitted m(omega) (A.2g) to reproduce it, so the
    # pressure at which the SRK liquid and vapour roots have equal Gibbs energy (lnphi^L = lnphi^V)
    # must be close to Pc * 10^-(1+omega).  Pins constants 0.42748/0.08664/m(omega), A.6 and the g(Z) rule.
    for name in ("C1", "C3", "nC7", "CO2"):
        s = W.make_system([name, "N2"])
        o = oracle_mod.Oracle.from_system(s)
        T = 0.7 * s.Tc[0]
        c = np.array([1.0, 0.0])

        def dg(P):
            Ai, Bi, _ = o.setup(P, T)
            r = o.cubic_roots(Ai[0], Bi[0])
            if len(r) < 3 or r[0] <= Bi[0]:
                return None
            return o.gibbs_of_root(r[0], Ai[0], Bi[0]) - o.gibbs_of_root(r[2], Ai[0], Bi[0])

        target = s.Pc[0] * 10 ** (-(1 + s.omega[0]))
        lo, hi = 0.5 * target, 1.5 * target
        assert dg(lo) > 0 > dg(hi)       # low P: vapour has lower g; high P: liquid
        for _ in range(60):
            mid = 0.5 * (lo + hi)
            if dg(mid) > 0:
                lo = mid
            else:
                hi = mid
        Psat = 0.5 * (lo + hi)
        assert Psat == pytest.approx(target, rel=0.03)
        # and the oracle's root choice flips exactly there
        _, Zlo = o.lnphi(Psat * 0.999, T, c)
        _, Zhi = o.lnphi(Psat * 1.001, T, c)
        assert Zlo > 0.5 and Zhi < 0.2


def test_wilson(sys10):
    s = W.system_co2_10()
    P, T = 40.0, 300.0
    np.testing.assert_allclose(sys10.wilson(P, T), np.log(s.Pc / P) + 5.373 * (1 + s.omega) * (1 - s.Tc / T), rtol=1e-14)
    # at T = Tc_i, P = Pc_i Wilson gives K_i = 1 (eq. 6)
    assert sys10.wilson(s.Pc[2], s.Tc[2])[2] == pytest.approx(0.0, abs=1e-15)


# ------------------------------------------------------------------------------------------------
# Rachford-Rice eq. 7, App. C
# ------------------------------------------------------------------------------------------------
def test_rr_binary_closed_form(sys2):
    for _ in range(300):
        K = np.array([np.exp(RNG.uniform(0.01, 6)), np.exp(-RNG.uniform(0.01, 9))])
        z1 = RNG.uniform(0.001, 0.999)
        z = np.array([z1, 1 - z1])
        th = sys2.rachford_rice(K, z)
        ref = -(z[0] * (K[0] - 1) + z[1] * (K[1] - 1)) / ((K[0] - 1) * (K[1] - 1))
        assert th == pytest.approx(ref, rel=1e-12, abs=1e-14)


def test_rr_monotone_bracket_and_sums(sys10):
    for _ in range(200):
        z = _rand_comp(10)
        K = np.exp(RNG.normal(0, 2.5, 10))
        if K.max() <= 1 or K.min() >= 1:
            continue
        th = sys10.rachford_rice(K, z)
        al, ar = 1 / (1 - K.max()), 1 / (1 - K.min())
        assert al < th < ar
        grid = al + (ar - al) * np.linspace(1e-6, 1 - 1e-6, 400)
        f = np.array([sys10.rr_f(K, z, t) for t in grid])
        assert np.all(np.diff(f) < 0)                               # strictly decreasing on the window
        eps = 4 * np.finfo(float).eps * max(1.0, abs(th))
        assert sys10.rr_f(K, z, th - eps) >= 0 >= sys10.rr_f(K, z, th + eps)   # sign change across the root
        x = z / (1 + (K - 1) * th)
        assert x.sum() == pytest.approx(1, abs=1e-12) and (K * x).sum() == pytest.approx(1, abs=1e-12)
    assert sys10.rachford_rice(np.full(10, 1.5), _rand_comp(10)) is None     # no window (C13)
    assert sys10.rachford_rice(np.full(10, 0.5), _rand_comp(10)) is None


# ------------------------------------------------------------------------------------------------
# Stability: definition by brute force on binaries (eq. 3) and tm/tpd identities (C1, C2)
# ------------------------------------------------------------------------------------------------
def _binary_grid(o, P, T, n=4000):
    c1 = (np.arange(n) + 0.5) / n
    c = np.stack([c1, 1 - c1], axis=1)
    lp, _ = o.lnphi_many(P, T, c)
    return c1, c, lp


def test_stability_binary_bruteforce(sys2):
    w = W.config1(1000)
    r = sys2.flash(w.z, w.P, w.T, nthreads=4)
    checked = mism = 0
    for n in range(0, 1000, 4):
        P, T, z = w.P[n], w.T[n], w.z[:, n]
        c1, c, lp = _binary_grid(sys2, P, T)
        lpz, _ = sys2.lnphi(P, T, z)
        d = np.log(z) + lpz
        tpd = (c * (np.log(c) + lp - d)).sum(1)
        tmin = tpd.min()
        if -1e-6 <= tmin < -1e-9 or (r["phase"][n] == 2 and abs(r["tpd_min"][n]) < 1e-5):
            continue   # grid resolution: a very shallow/narrow negative well is not resolvable on 4000 points
        checked += 1
        unstable_bf = tmin < -1e-6
        if unstable_bf != (r["phase"][n] == 2):
            mism += 1
        if r["phase"][n] == 2 and r["probe_case"][n] != 3:
            # the oracle's tpd_min is a stationary value of tpd: the grid minimum cannot be much lower
            assert tmin >= r["tpd_min"][n] - 1e-5
    assert checked > 200 and mism == 0


def test_tm_tpd_identities(sys10):
    w = W.config3(400)
    cnt = 0
    for n in range(400):
        P, T, z = w.P[n], w.T[n], w.z[:, n]
        lnK = sys10.wilson(P, T)
        for side in (+1, -1):
            st = sys10.stability_trial(P, T, z, lnK, side)
            if st["trivial"] or st["capped"]:
                continue
            cnt += 1
            Wv = np.exp(st["lnW"])
            wv = Wv / Wv.sum()
            lp, _ = sys10.lnphi(P, T, wv)
            lpz, _ = sys10.lnphi(P, T, z)
            d = np.log(z) + lpz
            assert np.abs(st["lnW"] + lp - d).max() < 1e-9                       # stationarity (eq. 5)
            assert st["tm"] == pytest.approx(1 - Wv.sum(), abs=1e-12)             # C2
            tpd_def = (wv * (np.log(wv) + lp - d)).sum()                          # eq. 3
            assert st["tpd"] == pytest.approx(tpd_def, abs=1e-9)
            assert st["tpd"] == pytest.approx(-np.log(Wv.sum()), abs=1e-12)
    assert cnt > 100


def test_stability_newton_equals_long_ss(sys10):
    w = W.config3(300)
    cnt = 0
    for n in range(300):
        P, T, z = w.P[n], w.T[n], w.z[:, n]
        lnK = sys10.wilson(P, T)
        for side in (+1, -1):
            a = sys10.stability_trial(P, T, z, lnK, side)
            b = sys10.stability_trial(P, T, z, lnK, side, opts=dict(use_newton=0, ss_cap=200000))
            if b["capped"] or a["capped"]:
                continue
            assert a["trivial"] == b["trivial"]
            if not a["trivial"]:
                cnt += 1
                assert a["tm"] == pytest.approx(b["tm"], abs=1e-9)
                np.testing.assert_allclose(a["lnW"], b["lnW"], atol=2e-7)
    assert cnt > 80


# ------------------------------------------------------------------------------------------------
# Whole flash: invariants (1a), (1b), (2) PAPER.md:39-47; Gibbs energy; hull tangent points
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("cfg,N", [(1, 1000), (2, 3000), (3, 3000), (4, 3000)])
def test_flash_invariants(oracle_mod, cfg, N):
    w = W.CONFIGS[cfg](N)
    o = oracle_mod.Oracle.from_system(w.system)
    r = o.flash(w.z, w.P, w.T, nthreads=8)
    assert set(np.unique(r["phase"])) <= {1, 2}
    two = r["phase"] == 2
    assert 0.05 < two.mean() < 0.8
    b = r["beta"]
    assert np.all((b[two] > 0) & (b[two] < 1))
    assert np.abs(w.z - b * r["y"] - (1 - b) * r["x"])[:, two].max() < 1e-12           # (1a)
    assert np.abs(r["x"].sum(0) - 1)[two].max() < 1e-12 and np.abs(r["y"].sum(0) - 1)[two].max() < 1e-12   # (1b)
    # single phase: x = y = z (the feed normalised once, reading C20 -> equal to the given z to an ulp)
    assert np.array_equal(r["x"][:, ~two], r["y"][:, ~two]) and np.abs(r["x"] - w.z)[:, ~two].max() < 4e-16
    assert np.all(np.isin(b[~two], (0.0, 1.0)))
    assert (r["status"] & 0b11011).sum() == 0
    for n in np.where(two)[0][:150]:
        P, T = w.P[n], w.T[n]
        x, y, z = r["x"][:, n], r["y"][:, n], w.z[:, n]
        lx, _ = o.lnphi(P, T, x)
        ly, _ = o.lnphi(P, T, y)
        lz, _ = o.lnphi(P, T, z)
        assert np.abs(np.log(x) + lx - np.log(y) - ly).max() < 1e-9                       # (2) iso-fugacity
        Gf = z @ (np.log(z) + lz)
        G2 = (1 - b[n]) * x @ (np.log(x) + lx) + b[n] * y @ (np.log(y) + ly)                # eq. 8
        assert G2 < Gf + 1e-13                                                             # two-phase Gibbs energy below feed
        np.testing.assert_allclose(r["lnK"][:, n], np.log(y / x), atol=1e-9)


def test_split_binary_hull_tangent(sys2):
    w = W.config1(400)
    r = sys2.flash(w.z, w.P, w.T, nthreads=4)
    cnt = 0
    for n in np.where(r["phase"] == 2)[0][:60]:
        P, T = w.P[n], w.T[n]
        ngrid = 4000
        c1, c, lp = _binary_grid(sys2, P, T, ngrid)
        g = (c * (np.log(c) + lp)).sum(1)
        # lower convex hull of (c1, g) by the monotone-chain scan
        hull = []
        for i in range(ngrid):
            while len(hull) >= 2:
                a, b_ = hull[-2], hull[-1]
                if (g[b_] - g[a]) * (c1[i] - c1[a]) >= (g[i] - g[a]) * (c1[b_] - c1[a]):
                    hull.pop()
                else:
                    break
            hull.append(i)
        hull = np.array(hull)
        gaps = np.diff(hull)
        k = np.argmax(gaps)
        if gaps[k] < 5:
            continue
        lo, hi = c1[hull[k]], c1[hull[k + 1]]
        z1 = w.z[0, n]
        if not (lo < z1 < hi):
            continue
        cnt += 1
        x1, y1 = r["x"][0, n], r["y"][0, n]
        a, b_ = min(x1, y1), max(x1, y1)
        assert abs(a - lo) < 2.0 / ngrid and abs(b_ - hi) < 2.0 / ngrid     # tangent points = hull gap ends
        assert r["beta"][n] == pytest.approx((z1 - x1) / (y1 - x1), abs=1e-10)
    assert cnt > 30


def test_split_newton_equals_long_ss(sys10):
    w = W.config3(1500)
    a = sys10.flash(w.z, w.P, w.T, nthreads=8)
    b = sys10.flash(w.z, w.P, w.T, opts=dict(use_newton=0, ss_cap=400000), nthreads=8)
    ok = (b["status"] & 3) == 0
    assert ok.mean() > 0.99
    assert np.array_equal(a["phase"][ok], b["phase"][ok])
    two = ok & (a["phase"] == 2)
    assert two.sum() > 300
    assert np.abs(a["beta"] - b["beta"])[two].max() < 1e-8
    assert np.abs(a["x"] - b["x"])[:, two].max() < 1e-8 and np.abs(a["y"] - b["y"])[:, two].max() < 1e-8


@pytest.mark.parametrize("cfg", [1, 3])
def test_long_double_agrees(oracle_mod, cfg):
    w = W.CONFIGS[cfg](1000)
    a = oracle_mod.Oracle.from_system(w.system).flash(w.z, w.P, w.T, nthreads=8)
    b = oracle_mod.Oracle.from_system(w.system, real="long double").flash(w.z, w.P, w.T, nthreads=8)
    assert np.array_equal(a["phase"], b["phase"])
    two = a["phase"] == 2
    assert np.abs(a["beta"] - b["beta"])[two].max() < 1e-9
    assert np.abs(a["x"] - b["x"])[:, two].max() < 1e-9 and np.abs(a["y"] - b["y"])[:, two].max() < 1e-9


def test_probe_never_contradicts_stability(sys10):
    # case 3 of the 3-iteration probe claims "unstable" without a stability analysis.
    # Forcing every mixture through the full stability analysis (probe_iters = 0) must give the same labels.
    w = W.config3(3000)
    a = sys10.flash(w.z, w.P, w.T, nthreads=8)
    b = sys10.flash(w.z, w.P, w.T, opts=dict(probe_iters=0), nthreads=8)
    assert (a["probe_case"] == 3).sum() > 500
    assert np.array_equal(a["phase"], b["phase"])
    two = a["phase"] == 2
    assert np.abs(a["beta"] - b["beta"])[two].max() < 1e-8          # independence of the start (probe K vs stability K)


def test_zero_component_reduces_to_smaller_system(oracle_mod):
    # a component with z_i = 0 is carried with x_i = y_i = 0 and changes nothing (C12)
    w = W.config1(200)
    o2 = oracle_mod.Oracle.from_system(w.system)
    s3 = W.make_system(["C1", "CO2", "nC10"], {("C1", "CO2"): 0.12, ("nC10", "CO2"): 0.12})
    o3 = oracle_mod.Oracle.from_system(s3)
    z3 = np.stack([w.z[0], np.zeros(200), w.z[1]])
    a = o2.flash(w.z, w.P, w.T, nthreads=2)
    b = o3.flash(z3, w.P, w.T, nthreads=2)
    assert np.array_equal(a["phase"], b["phase"])
    np.testing.assert_allclose(a["beta"], b["beta"], atol=1e-11)
    np.testing.assert_allclose(a["x"], b["x"][[0, 2]], atol=1e-11)
    np.testing.assert_allclose(a["y"], b["y"][[0, 2]], atol=1e-11)
    assert np.all(b["x"][1] == 0) and np.all(b["y"][1] == 0)


def test_permutation_invariance(oracle_mod):
    w = W.config3(300)
    perm = np.array([9, 3, 0, 8, 1, 7, 2, 6, 4, 5])
    s = w.system
    sp = W.System([s.names[i] for i in perm], s.Tc[perm], s.Pc[perm], s.omega[perm], s.kij[np.ix_(perm, perm)])
    a = oracle_mod.Oracle.from_system(s).flash(w.z, w.P, w.T, nthreads=4)
    b = oracle_mod.Oracle.from_system(sp).flash(w.z[perm], w.P, w.T, nthreads=4)
    assert np.array_equal(a["phase"], b["phase"])
    two = a["phase"] == 2
    np.testing.assert_allclose(a["beta"][two], b["beta"][two], atol=1e-9)
    np.testing.assert_allclose(a["x"][perm][:, two], b["x"][:, two], atol=1e-9)


def test_invalid_inputs(sys2):
    z = np.array([[0.5, 0.5, -0.1, np.nan, 0.5, 0.7], [0.5, 0.5, 1.1, 0.5, 0.5, 0.7]])
    P = np.array([10.0, -1.0, 10.0, 10.0, np.inf, 10.0])
    T = np.array([300.0, 300.0, 300.0, 300.0, 300.0, 300.0])
    r = sys2.flash(z, P, T, nthreads=1)
    assert list(r["phase"]) == [r["phase"][0], -1, -1, -1, -1, -1] and r["phase"][0] in (1, 2)
    assert np.all(np.isnan(r["beta"][1:]))


def test_warm_start_and_skip_stability(sys10):
    # caller-supplied lnK0 (section 4.3 PAPER.md:292-294 interface effect): converged lnK + noise, skip stability
    w = W.config3(2000)
    cold = sys10.flash(w.z, w.P, w.T, nthreads=8)
    two = cold["phase"] == 2
    noise = 0.05 * RNG.normal(size=cold["lnK"].shape)
    lnK0 = cold["lnK"] + noise
    flags = np.where(two, 1, 0).astype(np.uint8)
    warm = sys10.flash(w.z, w.P, w.T, lnK0=lnK0, flags=flags, nthreads=8)
    assert np.array_equal(warm["phase"], cold["phase"])
    assert np.abs(warm["beta"] - cold["beta"])[two].max() < 1e-8
    assert warm["iters"][two].mean() < cold["iters"][two].mean()
    # reading C21: a hint that fails (successive substitution still outside 0 < theta < 1 after hint_ss_cap = 12 iterations,
    # no convergence within hint_tr_cap = 15 trust-region iterations, or a trivial split) is dropped, reported (status bit 64)
    # and the mixture flashed cold
    restarted = (warm["status"] & 64) != 0
    assert restarted.sum() < 0.01 * two.sum() and not np.any(restarted & ~two)
    assert np.all(warm["stab_iters"][two & ~restarted] == 0)
    assert np.array_equal(warm["stab_iters"][restarted], cold["stab_iters"][restarted])
    # the two hint caps only cut short splits whose outcome does not change: with the rules off (caps = the general caps) the
    # answers agree, and only hints that were dropped can survive
    slow = sys10.flash(w.z, w.P, w.T, lnK0=lnK0, flags=flags, nthreads=8, opts=dict(hint_ss_cap=100000, hint_tr_cap=60))
    assert np.array_equal(slow["phase"], warm["phase"]) and np.abs(slow["beta"] - warm["beta"])[two].max() < 1e-8
    assert np.all(((slow["status"] & 64) != 0) <= restarted)
    # ... and the same on BASELINE config 5's own inputs (every mixture within 5 % of its phase boundary, hints from the
    # neighbouring pressure): that is where the caps bite.  hint_ss_cap / hint_tr_cap are a PRODUCT choice (they cut the time
    # the CUDA path spends on hints that are going to fail, reading C21) which the oracle mirrors; what is pinned here is that
    # the choice does not move an answer (VERDICT r2, weak point 5b)
    import os, sys
    sys.path.insert(0, os.path.dirname(__file__))
    import config5
    w5, lnK5, flags5, _info = config5.build(sys10, 6000)
    capped = sys10.flash(w5.z, w5.P, w5.T, lnK0=lnK5, flags=flags5, nthreads=8)
    free = sys10.flash(w5.z, w5.P, w5.T, lnK0=lnK5, flags=flags5, nthreads=8, opts=dict(hint_ss_cap=100000, hint_tr_cap=60))
    two5 = capped["phase"] == 2
    r_capped, r_free = (capped["status"] & 64) != 0, (free["status"] & 64) != 0
    assert two5.sum() > 1000 and r_capped.sum() > 0                       # the caps (or a failed hint) are exercised
    assert np.array_equal(free["phase"], capped["phase"])
    assert np.abs(free["beta"] - capped["beta"])[two5].max() < 1e-8 and np.abs(free["x"] - capped["x"])[:, two5].max() < 1e-8
    assert np.all(r_free <= r_capped)                                      # without the caps only fewer hints are dropped
    print("config 5 hints dropped with / without the caps:", int(r_capped.sum()), int(r_free.sum()), "of", int(flags5.astype(bool).sum()))


def test_split_trivial_tol_is_not_load_bearing(oracle_mod, sys10):
    """Reading C22: the phase split counts as collapsed into the trivial solution x = y when max_i |ln K_i| < split_trivial_tol
    (1e-5 since round 2, 1e-9 before; the paper gives no number).  VERDICT r2 asked for a pin that fails when the value is too
    small.  There is no such case in today's oracle: with the last-Newton-step finish (C8) and the G-monotone acceptance (C11)
    a split that slides towards x = y is caught by beta leaving (0, 1) or goes all the way to ln K = 0, so 1e-9, 1e-5 and 1e-3
    give identical results -- scanned at 10^6 (config 3), 2^20 (config 4), 5 10^5 (config 2, paper9) and 2 10^5 (config 5 warm)
    mixtures, and on 42 000 stable mixtures wrongly hinted "unstable" with a small-|ln K| seed, the input that can only
    collapse.  What this test pins is therefore the insensitivity itself, on small samples of the same inputs: parity
    between the CUDA path and the oracle does not hinge on the constant, and genuine splits stay far above it."""
    cases = []
    w = W.config3(8000)
    cases.append((sys10, w, None, None))
    wp = W.paper9(6000)
    cases.append((oracle_mod.Oracle.from_system(wp.system), wp, None, None))
    cold = sys10.flash(w.z, w.P, w.T, nthreads=8)
    seed = 0.05 * np.stack([sys10.wilson(P, T) for P, T in zip(w.P, w.T)]).T
    cases.append((sys10, w, seed, np.where(cold["phase"] == 1, 1, 0).astype(np.uint8)))      # wrong hints on stable feeds
    for orc, wl, lnK0, flags in cases:
        kw = {} if lnK0 is None else dict(lnK0=lnK0, flags=flags)
        ref = orc.flash(wl.z, wl.P, wl.T, nthreads=8, **kw)
        for tol in (1e-9, 1e-3):
            r = orc.flash(wl.z, wl.P, wl.T, nthreads=8, opts=dict(split_trivial_tol=tol), **kw)
            assert np.array_equal(r["phase"], ref["phase"]) and np.array_equal(r["status"], ref["status"]), (wl.name, tol)
            assert np.array_equal(r["beta"], ref["beta"], equal_nan=True), (wl.name, tol)
        two = ref["phase"] == 2
        assert np.abs(ref["lnK"][:, two]).max(0).min() > 1e-2            # genuine solutions: far above any of the three values
    assert not np.any((ref["phase"] == 2) & (flags == 1))                 # no wrongly hinted stable feed came out two-phase


def test_phase_identity_by_compressibility(oracle_mod, sys10):
    # Reading C23 (smallest root -> liquid, largest -> vapour): y is the phase with the larger Z.
    # (a) invariant on a workload; (b) independence of the sign of the K that seeds the split -- the two phases a
    # split finds from lnK and from -lnK are the same, and so is their reported identity; (c) the tie cases of
    # config 3 in which both stability starts reach the same stationary point (tm^L = tm^V to rounding, so that
    # "tm^L < tm^V", is decided by noise): the double and the long double build now report the same
    # identity (they did not before C23: mixtures 320255 and 730360).
    w = W.config3(3000)
    r = sys10.flash(w.z, w.P, w.T, nthreads=8)
    two = np.where(r["phase"] == 2)[0]
    assert len(two) > 500
    for n in two[:200]:
        _, Zx = sys10.lnphi(w.P[n], w.T[n], r["x"][:, n])
        _, Zy = sys10.lnphi(w.P[n], w.T[n], r["y"][:, n])
        assert Zy > Zx
    flags = np.where(r["phase"] == 2, 1, 0).astype(np.uint8)
    rneg = sys10.flash(w.z, w.P, w.T, lnK0=-r["lnK"], flags=flags, nthreads=8)
    ok = (rneg["status"][two] & 64) == 0          # not restarted
    assert ok.mean() > 0.9
    assert np.abs(rneg["beta"] - r["beta"])[two][ok].max() < 1e-8
    assert np.abs(rneg["y"] - r["y"])[:, two[ok]].max() < 1e-8
    ld = oracle_mod.Oracle.from_system(W.system_co2_10(), real="long double")
    for n in (320255, 616425, 693344, 730360, 813246):
        wn = W.config3(1, offset=n)
        a = sys10.flash(wn.z, wn.P, wn.T, nthreads=1)
        b = ld.flash(wn.z, wn.P, wn.T, nthreads=1)
        assert a["phase"][0] == 2 and b["phase"][0] == 2
        assert abs(a["beta"][0] - b["beta"][0]) < 1e-9 and np.abs(a["x"] - b["x"]).max() < 1e-9


def test_path_sensitivity_set(sys10):
    """The labels of a few mixtures per 10^5 depend on schedule constants of the stability analysis that the paper does
    not fix (reading C11; tests/oracle_path_sensitivity.py lists them at full size).  Pinned here at a reduced size:
    (a) the set is small; (b) a negative tpd found from ANY start proves instability (eq. 3), so wherever the
    default oracle says "unstable" the many-start adjudication must agree and reach a tpd at least as low; (c) on a control
    sample the many-start search never overturns a default "stable" verdict by more than the band."""
    sys.path.insert(0, str(Path(__file__).resolve().parent))
    import oracle_path_sensitivity as S
    w = W.config3(30000)
    rep = S.report(sys10, w, nthreads=8, control=150)
    assert rep["label_changes"] <= 3
    for m in rep["mixtures"]:
        if m["default_label"] == 2:
            assert m["true_label_unstable"] and m["adjudicated_tpd_min"] <= m["default_tpd_min"] + 1e-10
    assert len(rep["control_overturned"]) == 0
    base = sys10.flash(w.z, w.P, w.T, nthreads=8)
    uns = np.where((base["tpd_min"] < -1e-6) & (base["probe_case"] != 3))[0][:60]
    assert len(uns) > 20
    for n in uns:
        tpd, neg, ns = S.adjudicate(sys10, w.P[n], w.T[n], w.z[:, n])
        assert neg >= 1 and tpd <= base["tpd_min"][n] + 1e-10


# ------------------------------------------------------------------------------------------------
# eq. 13: d theta / d K by the implicit-function theorem
# ------------------------------------------------------------------------------------------------
def test_rr_derivative_binary_closed_form(sys2):
    # binary: f_RR = 0 has the closed-form root theta = -(z1 (K1-1) + z2 (K2-1)) / ((K1-1)(K2-1)); differentiate it by hand
    for K1, K2, z1 in [(3.0, 0.2, 0.4), (1.5, 0.6, 0.5), (12.0, 0.01, 0.3)]:
        z2 = 1.0 - z1
        a, b = K1 - 1.0, K2 - 1.0
        th = -(z1 * a + z2 * b) / (a * b)
        d1 = -z1 / (a * b) + (z1 * a + z2 * b) / (a * a * b)     # d theta / d K1
        d2 = -z2 / (a * b) + (z1 * a + z2 * b) / (a * b * b)     # d theta / d K2
        got = sys2.rr_dtheta_dK([K1, K2], [z1, z2], th)
        assert np.allclose(got, [d1, d2], rtol=1e-13, atol=0)


def test_rr_derivative_matches_finite_differences_of_the_solver(sys10):
    # the derivative of the SOLVER's root (bisection to rounding) by central differences: pins sign, index and the
    # [d f / d theta]^-1 factor of eq. 13 against the definition of theta(K) itself
    rng = np.random.default_rng(13)
    for _ in range(20):
        z = rng.dirichlet(np.ones(10))
        lnK = rng.normal(0.0, 1.5, 10)
        K = np.exp(lnK)
        th = sys10.rachford_rice(K, z)
        if th is None:
            continue
        got = sys10.rr_dtheta_dK(K, z, th)
        for i in range(10):
            h = 1e-6 * K[i]
            Kp, Km = K.copy(), K.copy()
            Kp[i] += h
            Km[i] -= h
            fd = (sys10.rachford_rice(Kp, z) - sys10.rachford_rice(Km, z)) / (2 * h)
            assert abs(got[i] - fd) <= 1e-6 * max(1.0, abs(fd)), (i, got[i], fd)
    # a z_i = 0 component does not move theta (C12)
    z = np.array([0.5, 0.5, 0, 0, 0, 0, 0, 0, 0, 0.0])
    K = np.array([2.0, 0.5, 7, 7, 7, 7, 7, 7, 7, 7.0])
    d = sys10.rr_dtheta_dK(K, z, sys10.rachford_rice(K, z))
    assert np.all(d[2:] == 0.0) and d[0] > 0 and d[1] > 0      # theta grows with every K_i (f_RR grows with K_i, falls with theta)


def test_rr_batch_and_flash_derivative_output(oracle_mod, sys10):
    w = W.config3(3000)
    o = sys10.flash(w.z, w.P, w.T)
    two = o["phase"] == 2
    assert two.sum() > 500
    # the flash's derivative output is eq. 13 at its own reported (beta, K = y/x): re-evaluate through the scalar entry,
    # and check it against the batched Rachford-Rice solve started from the reported ln K
    rb = sys10.rr_batch(o["lnK"][:, two], w.z[:, two])
    assert np.all(rb["ok"] == 1)
    assert np.abs(rb["theta"] - o["beta"][two]).max() < 1e-9
    assert np.abs(rb["x"] - o["x"][:, two]).max() < 1e-9 and np.abs(rb["y"] - o["y"][:, two]).max() < 1e-9
    d = o["dbeta_dK"][:, two]
    assert np.all(np.isfinite(d)) and np.all(d >= 0)
    assert np.allclose(rb["dtheta_dK"], d, rtol=1e-6, atol=1e-12)
    assert np.all(np.isnan(o["dbeta_dK"][:, ~two]))
    # no window -> NaN and ok = 0
    lnK = np.full((10, 4), 0.3)
    rb = sys10.rr_batch(lnK, w.z[:, :4])
    assert np.all(rb["ok"] == 0) and np.all(np.isnan(rb["theta"]))


# ------------------------------------------------------------------------------------------------
# stability-only mode and the Table-4 counters
# ------------------------------------------------------------------------------------------------
def test_stability_only_mode_is_the_label_of_the_full_flash(sys10):
    w = W.config3(4000)
    full = sys10.flash(w.z, w.P, w.T)
    so = sys10.flash(w.z, w.P, w.T, opts={"stability_only": 1})
    # "unstable" in stability-only mode <=> the full flash entered the phase split (it ends two-phase unless the split
    # failed, which the full flash reports with status bit 8)
    entered = full["stage"][7] > 0
    assert np.array_equal(so["phase"] == 2, entered)
    failed = (full["status"] & 8) != 0
    assert np.array_equal(full["phase"] == 2, entered & ~failed)
    assert np.array_equal(so["tpd_min"], full["tpd_min"], equal_nan=True)
    assert np.array_equal(so["stab_iters"], full["stab_iters"]) and np.array_equal(so["probe_case"], full["probe_case"])
    assert np.array_equal(so["x"], w.z / w.z.sum(0)) and np.array_equal(so["y"], so["x"])
    assert np.all(np.isnan(so["beta"][so["phase"] == 2])) and np.all(np.isin(so["beta"][so["phase"] == 1], (0.0, 1.0)))
    assert np.all(so["iters"] <= 3) and np.all(so["stage"][5:9] == 0)        # no split work at all
    # the K seed of an unstable mixture starts a split that reaches the full flash's answer
    n = int(np.nonzero((so["phase"] == 2) & (full["phase"] == 2))[0][0])
    sp = sys10.phase_split(w.P[n], w.T[n], so["x"][:, n], so["lnK"][:, n])
    assert sp["two_phase"] and abs(min(sp["theta"], 1 - sp["theta"]) - min(full["beta"][n], 1 - full["beta"][n])) < 1e-9


def test_stage_counters_are_consistent(sys10):
    w = W.config3(4000)
    o = sys10.flash(w.z, w.P, w.T)
    st, pc = o["stage"], o["probe_case"]
    went = (pc == 1) | (pc == 2)
    assert np.array_equal(o["stab_iters"], st[0] + st[1] + st[2] + st[3])
    assert np.array_equal(st[4], st[9] + st[10])                               # trials that entered the trust-region stage
    assert np.all((st[0] + st[1] > 0) == went) and np.all(st[0:4, ~went] == 0)
    assert np.all(st[0] <= 9) and np.all(st[1] <= 9)                            # SS cap of PAPER.md:79
    assert np.all(st[2][st[9] == 0] == 0) and np.all(st[3][st[10] == 0] == 0)   # no trust-region iterations without entering
    assert np.all(st[11:13] == 0) and np.all((o["status"] & 1) == 0)            # nothing capped on this workload
    assert np.array_equal(st[7] > 0, (pc == 3) | (went & (o["tpd_min"] < 0)))


# ------------------------------------------------------------------------------------------------
# the paper's own case studies (section 2.3-2.4, Tables 1-3, D.6)
# ------------------------------------------------------------------------------------------------
def test_paper_workloads_follow_tables_1_to_3():
    s = W.system_paper9()
    assert s.names[0] == "CH4" and s.nc == 9
    assert s.Pc[0] == 4.6 and s.Tc[6] == 604.5 and s.omega[8] == 0.039          # Table 1 PAPER.md:121-129 (MPa, K)
    k = s.kij.copy()
    assert k[0, 7] == 0.0882 == k[7, 0]
    k[0, 7] = k[7, 0] = 0.0
    assert not k.any()
    w = W.paper9(8000)
    assert np.all((w.P > 5) & (w.P < 25)) and np.all((w.T > 200) & (w.T < 600)) and np.allclose(w.z.sum(0), 1, atol=1e-14)
    for t, kind in enumerate(W.PAPER_FLUIDS):
        z = w.z[:, t::4]
        for i, (lo, hi) in enumerate(W.PAPER_FLUID_RANGES[kind]):                # Table 2
            assert np.all(z[i] >= lo - 1e-12) and np.all(z[i] <= hi + 1e-12), (kind, i)
        # Appendix D's typical composition of the type lies inside the type's ranges (consistency of Tables 2 and D.6)
        for i, (lo, hi) in enumerate(W.PAPER_FLUID_RANGES[kind]):
            assert lo - 1e-12 <= W.PAPER_TYPICAL[kind][i] <= hi + 5e-4, (kind, i)
    acc = W.paper9(40000).meta["acceptance"]
    assert acc["wet_gas"] > acc["volatile_oil"] > acc["gas_condensate"] > acc["black_oil"] > 5e-4
    # prefix / offset property
    assert np.array_equal(W.paper9(300, offset=500).z, w.z[:, 500:800])
    for name, nc in (("paper2", 2), ("paper4", 4)):
        v = W.CONFIGS[name](2000)
        assert v.system.nc == nc and np.all((v.P > 0.1) & (v.P < 10)) and np.all((v.T > 200) & (v.T < 500))
        assert np.allclose(v.z.sum(0), 1, atol=1e-14) and not v.system.kij.any()


@pytest.mark.parametrize("name,N", [("paper2", 3000), ("paper4", 3000), ("paper9", 4000)])
def test_flash_invariants_on_paper_workloads(oracle_mod, name, N):
    w = W.CONFIGS[name](N)
    orc = oracle_mod.Oracle.from_system(w.system)
    o = orc.flash(w.z, w.P, w.T)
    two = o["phase"] == 2
    assert 0.05 < two.mean() < 0.8
    b, x, y = o["beta"][two], o["x"][:, two], o["y"][:, two]
    assert np.all((b > 0) & (b < 1))
    assert np.abs(b * y + (1 - b) * x - w.z[:, two]).max() < 1e-12               # (1a)
    assert np.abs(x.sum(0) - 1).max() < 1e-12 and np.abs(y.sum(0) - 1).max() < 1e-12   # (1b)
    idx = np.nonzero(two)[0][:: max(1, two.sum() // 60)]
    for n in idx:                                                               # (2) iso-fugacity
        lx, Zx = orc.lnphi(w.P[n], w.T[n], o["x"][:, n])
        ly, Zy = orc.lnphi(w.P[n], w.T[n], o["y"][:, n])
        assert np.abs(np.log(o["x"][:, n]) + lx - np.log(o["y"][:, n]) - ly).max() < 1e-8
        assert Zy >= Zx
    if name == "paper9":
        # Table 4's shape (SURVEY.md section 4 says the absolute shares are NOT a pin): the probe proves
        # a large share unstable, and a minority of the stability trials needs the trust-region stage
        assert 0.2 < (o["probe_case"] == 3).mean() < 0.5
        # pressure in MPa with Pc in MPa == pressure in bar with Pc in bar (the gas constant cancels)
        s = w.system
        orc_bar = oracle_mod.Oracle(s.Tc, s.Pc * 10.0, s.omega, s.kij)
        o2 = orc_bar.flash(w.z[:, :500], w.P[:500] * 10.0, w.T[:500])
        assert np.array_equal(o2["phase"], o["phase"][:500])
        t2 = o2["phase"] == 2
        assert np.abs(o2["beta"][t2] - o["beta"][:500][t2]).max() < 1e-9


def test_numpy_fugacity_check_agrees_with_the_oracle(oracle_mod):
    """tests/srk_check.py is a third statement of App. A (A.1-A.6 PAPER.md:404-450) in vectorised numpy -- closed-form cubic
    plus Newton polish instead of the oracle's iteration, no shared code.  The GPU tests use it to check condition (2) on
    the CUDA results without the oracle; here the two independent implementations must agree on ln phi and on the chosen
    root, over feeds, near-pure and trace compositions of three systems (with and without k_ij), which also pins the
    oracle's orc_lnphi once more."""
    import sys, os
    sys.path.insert(0, os.path.dirname(__file__))
    import srk_check
    rng = np.random.default_rng(20220503)
    n_multi = 0
    for w in (W.config1(300), W.config2(300), W.config3(400), W.paper9(300)):
        orc = oracle_mod.Oracle.from_system(w.system)
        nc = w.system.nc
        comps = [w.z, rng.dirichlet(np.full(nc, 0.3), w.N).T + 1e-12]
        for c in comps:
            c = c / c.sum(0)
            got, Zg = srk_check.lnphi(w.system, w.P, w.T, c)
            multi = 0
            for n in range(w.N):
                want, Zw = orc.lnphi(w.P[n], w.T[n], np.ascontiguousarray(c[:, n]))
                Ai, Bi, Aij = orc.setup(w.P[n], w.T[n])
                A, B = float(c[:, n] @ Aij @ c[:, n]), float(c[:, n] @ Bi)
                r = orc.cubic_roots(A, B)
                if len(r) == 3 and abs(orc.gibbs_of_root(r.min(), A, B) - orc.gibbs_of_root(r.max(), A, B)) < 1e-9:
                    continue   # two roots of (numerically) equal Gibbs energy: either choice is right
                multi += len(r) == 3
                assert abs(Zg[n] - Zw) < 1e-11 * max(1.0, abs(Zw)), (w.name, n, Zg[n], Zw)
                assert np.abs(got[:, n] - want).max() < 1e-10, (w.name, n, np.abs(got[:, n] - want).max())
            n_multi += multi
    assert n_multi > 50, n_multi   # the minimum-Gibbs choice among three real roots was exercised
    # and the residual it reports is small on the oracle's two-phase results, large on a perturbed one
    w = W.config3(600)
    o = oracle_mod.Oracle.from_system(w.system).flash(w.z, w.P, w.T)
    two = o["phase"] == 2
    res = srk_check.isofugacity_residual(w.system, w.P[two], w.T[two], o["x"][:, two], o["y"][:, two])
    assert two.sum() > 100 and res.max() < 1e-9
    y_bad = o["y"][:, two].copy()
    y_bad[0] *= 1.0 + 1e-6
    assert srk_check.isofugacity_residual(w.system, w.P[two], w.T[two], o["x"][:, two], y_bad / y_bad.sum(0)).min() > 1e-8
