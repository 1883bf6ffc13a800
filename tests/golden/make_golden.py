"""Writes the stored expected values under tests/golden/ that are not printed in the paper itself.

  python tests/golden/make_golden.py

Calls neither the CUDA path nor (for these two files) the oracle: the values come from scipy's exponential
integral and from exact decimal arithmetic, so that they pin the oracle / the input recipe from outside.

diffusivity_eq7.txt   D(dtau) = -ln(T)/dtau with T = (1 - dtau) e^-dtau + dtau^2 E1(dtau) = 2 E3(dtau)
                      (eq. 6-7; Fig. 1 at PAPER.md:177), T from scipy.special.expn(3, .).
rayleigh_h2.txt       sigma_scat of eq. 16 with n_ref = 2.68678e19 cm^-3, K = 1 and n_lambda of eq. 17
                      (PAPER.md:195-206), in 40-digit decimal arithmetic, and sigma / (2.4 m_p).
"""
import decimal
import os

import numpy as np
from scipy import special

HERE = os.path.dirname(os.path.abspath(__file__))


def diffusivity():
    rows = []
    for dtau in (1e-3, 1e-2, 0.1, 0.5, 1.0, 2.0, 10.0, 30.0):
        T = 2.0 * special.expn(3, dtau)
        rows.append((dtau, -np.log(T) / dtau))
    with open(os.path.join(HERE, "diffusivity_eq7.txt"), "w") as f:
        f.write("# Exact diffusivity factor of eq. 7 (PAPER.md:111): D = -ln(T)/dtau, T = 2 E3(dtau) (eq. 6, PAPER.md:105-107).\n"
                "# Written by tests/golden/make_golden.py from scipy.special.expn; Fig. 1 (PAPER.md:177): D -> 2 for thin,\n"
                "# D -> 1 for thick layers.  columns: dtau  D\n")
        for dtau, D in rows:
            f.write(f"{dtau:g} {D:.7f}\n")


def rayleigh():
    decimal.getcontext().prec = 40
    Dm = decimal.Decimal
    pi = Dm("3.141592653589793238462643383279502884197")
    n_ref = Dm("2.68678e19")
    m_p = Dm("1.67262192369e-24")                       # g, CODATA 2018
    mbar = Dm("2.4") * m_p
    rows = []
    for lam_um in ("0.3", "0.5", "1.0", "2.0"):
        lam = Dm(lam_um) * Dm("1e-4")                   # cm
        n = Dm("13.58e-5") * (1 + Dm("7.52e-11") / (lam * lam)) + 1       # eq. 17
        r = (n * n - 1) / (n * n + 2)
        sigma = 24 * pi ** 3 / (n_ref ** 2 * lam ** 4) * r * r            # eq. 16, K = 1
        rows.append((lam_um, sigma, sigma / mbar))
    with open(os.path.join(HERE, "rayleigh_h2.txt"), "w") as f:
        f.write("# Rayleigh cross-section of H2, eq. 16-17 (PAPER.md:195-206; n_ref = 2.68678e19 cm^-3, K = 1), and the\n"
                "# scattering opacity sigma/(2.4 m_p) (PAPER.md:208, 220; m_p = 1.67262192369e-24 g), 40-digit decimal\n"
                "# arithmetic, written by tests/golden/make_golden.py.  columns: lambda[um]  sigma[cm^2]  kappa_scat[cm^2/g]\n")
        for lam_um, s, k in rows:
            f.write(f"{lam_um} {s:.12e} {k:.12e}\n")


if __name__ == "__main__":
    diffusivity()
    rayleigh()
