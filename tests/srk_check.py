"""A third, independent statement of the SRK fugacity coefficients (App. A, A.1-A.6 at lines 404-450), in
vectorised numpy, used by the GPU tests to check the iso-fugacity condition (2) on the CUDA results
WITHOUT going through the oracle (parity against the oracle cannot see an error both sides share).

Test infrastructure only.  It shares no code with oracle/ or with the CUDA path; tests/test_oracle_pins.py pins it
against the oracle's ln phi (two independent implementations agreeing to 1e-11), which is also one more pin of the
oracle."""
import numpy as np


def lnphi(system, P, T, c):
    """ln phi_i of mixtures of composition c [nc, M] at P [M], T [M] -> (lnphi [nc, M], Z [M]).

    A.2: a_i, b_i from (Tc, Pc, omega), alpha_i = (1 + m_i (1 - sqrt(T / Tc_i)))^2, van der Waals mixing with k_ij;
    A.3: Z^3 - Z^2 + (A - B - B^2) Z - A B = 0; of several real roots above B the one of minimum Gibbs energy (A.5);
    A.6: ln phi_i = B_i/B (Z - 1) - ln(Z - B) - A/B (2 S_i / A - B_i / B) ln(1 + B / Z), S_i = sum_j c_j sqrt(A_i A_j)(1 - k_ij)."""
    Tc, Pc, om = (np.asarray(a, float)[:, None] for a in (system.Tc, system.Pc, system.omega))
    kij = np.zeros((len(system.Tc),) * 2) if system.kij is None else np.asarray(system.kij, float)
    P, T, c = np.asarray(P, float)[None, :], np.asarray(T, float)[None, :], np.asarray(c, float)
    m = 0.480 + 1.574 * om - 0.176 * om ** 2
    alpha = (1.0 + m * (1.0 - np.sqrt(T / Tc))) ** 2
    Ai = 0.42748 * alpha * (P / Pc) / (T / Tc) ** 2          # a_i P / (R T)^2: the gas constant cancels
    Bi = 0.08664 * (P / Pc) / (T / Tc)                       # b_i P / (R T)
    sA = np.sqrt(Ai)
    S = sA * ((1.0 - kij) @ (c * sA))
    A = (c * S).sum(0)
    B = (c * Bi).sum(0)
    c1 = A - B - B * B
    c0 = -A * B
    # depressed cubic t^3 + p t + q = 0, Z = t + 1/3
    p = c1 - 1.0 / 3.0
    q = -2.0 / 27.0 + c1 / 3.0 + c0
    disc = 0.25 * q * q + p * p * p / 27.0
    M = A.shape[0]
    roots = np.full((3, M), np.nan)
    one = disc > 0
    sq = np.sqrt(np.where(one, disc, 0.0))
    roots[0] = np.where(one, np.cbrt(-0.5 * q + sq) + np.cbrt(-0.5 * q - sq) + 1.0 / 3.0, np.nan)
    three = ~one
    pp = np.where(three, np.minimum(p, -1e-300), -1.0)
    r = 2.0 * np.sqrt(-pp / 3.0)
    arg = np.clip(3.0 * q / (pp * r), -1.0, 1.0)
    phi = np.arccos(arg)
    for k in range(3):
        t = r * np.cos((phi - 2.0 * np.pi * k) / 3.0)
        roots[k] = np.where(three, t + 1.0 / 3.0, roots[k])
    # the closed form loses digits by cancellation: three Newton steps on the cubic itself
    for _ in range(3):
        f = ((roots - 1.0) * roots + c1) * roots + c0
        df = (3.0 * roots - 2.0) * roots + c1
        roots = roots - np.where(np.abs(df) > 1e-300, f / np.where(df == 0, 1.0, df), 0.0)
    valid = np.isfinite(roots) & (roots > B)
    with np.errstate(invalid="ignore", divide="ignore"):
        gibbs = roots - 1.0 - np.log(np.where(valid, roots - B, 1.0)) - (A / B) * np.log1p(B / np.where(valid, roots, 1.0))
    gibbs = np.where(valid, gibbs, np.inf)
    Z = roots[np.argmin(gibbs, axis=0), np.arange(M)]
    out = Bi / B * (Z - 1.0) - np.log(Z - B) - (A / B) * (2.0 * S / A - Bi / B) * np.log1p(B / Z)
    return out, Z


def isofugacity_residual(system, P, T, x, y):
    """max_i |ln x_i + ln phi_i(x) - ln y_i - ln phi_i(y)| per mixture, over the components present (x_i, y_i > 0)."""
    lx, _ = lnphi(system, P, T, x)
    ly, _ = lnphi(system, P, T, y)
    present = (x > 0) & (y > 0)
    with np.errstate(divide="ignore", invalid="ignore"):
        r = np.where(present, np.log(x) + lx - np.log(y) - ly, 0.0)
    return np.abs(r).max(0)
