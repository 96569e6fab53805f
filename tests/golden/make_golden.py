"""Writes the closed-form fixtures of this directory.  Calls neither oracle/ nor the CUDA path: every number is a
textbook closed form evaluated with mpmath at 40 digits and rounded once (citations in each file's header).

    python tests/golden/make_golden.py
"""
import os

import mpmath as mp

mp.mp.dps = 40
HERE = os.path.dirname(os.path.abspath(__file__))


def fmt(x):
    return mp.nstr(x, 20)


def eigenvalues():
    out = ["# Eigenvalues of A = I + sigma (delta^2)^2 = circulant(sigma, -4 sigma, 1 + 6 sigma, -4 sigma, sigma) on N points:",
           "# lambda_k = 1 + sigma (2 - 2 cos(2 pi k / N))^2   (textbook circulant; SURVEY.md section 8(c); scheme P:522, north star)",
           "# columns: N sigma k lambda_k"]
    for N in (8, 16):
        for sigma in ("0.01", "1", "529"):
            for k in range(N // 2 + 1):
                lam = 1 + mp.mpf(sigma) * (2 - 2 * mp.cos(2 * mp.pi * k / N)) ** 2
                out.append(f"{N} {sigma} {k} {fmt(lam)}")
    open(os.path.join(HERE, "circulant_eigenvalues.txt"), "w").write("\n".join(out) + "\n")


def growth():
    out = ["# Linear growth factor of one Fourier mode C = cbar + eps cos(theta . i), theta_d = 2 pi m_d / N, per step of",
           "# Prod_d (I + gamma dt L_d) dC = dt Lap_h [(3 cbar^2 - 1) C - gamma Lap_h C]  (eq. (3) P:29-30 linearised; scheme P:522, north star):",
           "# g = 1 - dt S [(3 cbar^2 - 1) + gamma S] / Prod_d (1 + gamma dt s_d^2),  s_d = 2 - 2 cos theta_d,  S = sum_d s_d",
           "# columns: D N m_x m_y m_z cbar gamma dt g"]
    cases = [(2, 16, 3, 1, 0, "0", "1", "0.01"), (2, 16, 3, 1, 0, "-0.4", "1", "0.01"), (2, 64, 5, 9, 0, "0.3", "0.5", "0.02"),
             (3, 8, 1, 2, 3, "0", "1", "0.01"), (3, 16, 2, 5, 7, "-0.4", "2", "0.005"), (2, 32, 1, 1, 0, "0", "66.4", "7.97")]
    for D, N, mx, my, mz, cbar, gamma, dt in cases:
        ms = (mx, my, mz)[:D]
        s = [2 - 2 * mp.cos(2 * mp.pi * m / N) for m in ms]
        S = sum(s)
        cb, g_, d_ = mp.mpf(cbar), mp.mpf(gamma), mp.mpf(dt)
        den = mp.mpf(1)
        for sd in s:
            den *= 1 + g_ * d_ * sd ** 2
        g = 1 - d_ * S * ((3 * cb ** 2 - 1) + g_ * S) / den
        out.append(f"{D} {N} {mx} {my} {mz} {cbar} {gamma} {dt} {fmt(g)}")
    open(os.path.join(HERE, "growth_factors.txt"), "w").write("\n".join(out) + "\n")


def kink():
    out = ["# Energy per unit length of the stationary interface C = tanh(x / sqrt(2 gamma)) of eq. (3), P:29-30, with",
           "# F = int [ (C^2 - 1)^2 / 4 + gamma |grad C|^2 / 2 ]  (eq. (4), P:34, with the 1/4 of reading G3): (2 sqrt 2 / 3) sqrt gamma",
           "# columns: gamma energy_per_unit_length"]
    for gamma in ("1", "0.25", "0.01"):
        out.append(f"{gamma} {fmt(2 * mp.sqrt(2) / 3 * mp.sqrt(mp.mpf(gamma)))}")
    open(os.path.join(HERE, "kink_energy.txt"), "w").write("\n".join(out) + "\n")


def dissipation():
    out = ["# Leading-order dissipation of one Fourier mode C = cbar + eps cos(theta . i), theta_d = 2 pi m_d / N (eq. (4) P:34, eq. (6) P:64,",
           "# readings G4/G5): mu = mubar + eps K cos(theta . i) + O(eps^2), K = (3 cbar^2 - 1) + gamma S, and with forward differences",
           "# sum_i (mu_{i+e_d} - mu_i)^2 = eps^2 K^2 (N^D / 2) s_d, so  Fdot = - eps^2 K^2 (N^D / 2) sum_d s_d,  s_d = 2 - 2 cos theta_d, S = sum_d s_d.",
           "# Each axis contributes its own s_d (all distinct below): a dropped, duplicated or swapped axis term changes the value.",
           "# columns: D N m_x m_y m_z cbar gamma eps Fdot_leading per_axis_terms(x y z)"]
    cases = [(3, 8, 1, 2, 3, "0", "1", "1e-5"), (3, 16, 2, 5, 7, "-0.4", "2", "1e-6"), (3, 12, 1, 4, 5, "0.3", "0.5", "1e-6"),
             (2, 16, 3, 1, 0, "0", "1", "1e-5"), (2, 32, 5, 9, 0, "-0.4", "0.7", "1e-6")]
    for D, N, mx, my, mz, cbar, gamma, eps in cases:
        ms = (mx, my, mz)[:D]
        s = [2 - 2 * mp.cos(2 * mp.pi * m / N) for m in ms]
        S = sum(s)
        cb, g_, e_ = mp.mpf(cbar), mp.mpf(gamma), mp.mpf(eps)
        K = (3 * cb ** 2 - 1) + g_ * S
        terms = [-e_ ** 2 * K ** 2 * mp.mpf(N) ** D / 2 * sd for sd in s] + [mp.mpf(0)] * (3 - D)
        out.append(f"{D} {N} {mx} {my} {mz} {cbar} {gamma} {eps} {fmt(sum(terms))} " + " ".join(fmt(t) for t in terms))
    open(os.path.join(HERE, "mode_dissipation.txt"), "w").write("\n".join(out) + "\n")


if __name__ == "__main__":
    eigenvalues(); growth(); kink(); dissipation()
