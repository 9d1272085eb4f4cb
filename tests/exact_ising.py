"""Exact results for the 2D Ising model used to PIN the oracle (test-only; independent of oracle/ and of
the CUDA path).  Nothing here is taken from either implementation.

* kaufman_lnZ: B. Kaufman's closed form (Phys. Rev. 76, 1232 (1949)) for the L x L periodic lattice -- the
  finite-lattice partition function from which Beale's exact density of states is derived (BASELINE.json
  north_star "Beale's exact finite-L partition function"); SURVEY.md section 8(c) states the formula.
* onsager_lnZ_per_site: thermodynamic limit (Onsager 1944).
* brute_force_dos: density of states by enumerating all 2^N states with a numpy-roll energy (definition
  PAPER.md:78 eq. 6 written a second, vectorised way).
"""
import numpy as np
from mpmath import mp, mpf, cosh, sinh, tanh, acosh, log, cos, pi, quad, sqrt, exp


def kaufman_lnZ(L, beta, dps=60):
    mp.dps = dps
    K = mpf(beta)
    if K == 0:
        return L * L * log(2)
    N = L * L

    def gamma(l):
        if l == 0:
            return 2 * K + log(tanh(K))
        c = cosh(2 * K) * (cosh(2 * K) / sinh(2 * K)) - cos(l * pi / L)
        return acosh(c)

    Z1 = Z2 = Z3 = Z4 = mpf(1)
    for r in range(L):
        g_odd = gamma(2 * r + 1)
        g_even = gamma(2 * r)
        Z1 *= 2 * cosh(L * g_odd / 2)
        Z2 *= 2 * sinh(L * g_odd / 2)
        Z3 *= 2 * cosh(L * g_even / 2)
        Z4 *= 2 * sinh(L * g_even / 2)
    Z = (2 * sinh(2 * K)) ** (mpf(N) / 2) * (Z1 + Z2 + Z3 + Z4) / 2
    return log(Z)


def onsager_lnZ_per_site(beta, dps=40):
    mp.dps = dps
    K = mpf(beta)
    kappa = 2 * sinh(2 * K) / cosh(2 * K) ** 2
    integral = quad(lambda phi: log((1 + sqrt(1 - kappa ** 2 * mp.sin(phi) ** 2)) / 2), [0, pi])
    return log(2 * cosh(2 * K)) + integral / (2 * pi)


def brute_force_dos(L):
    """{E: count} over all 2^(L*L) states; energy = -sum over bonds (right and down neighbour) of s*s'."""
    N = L * L
    assert N <= 20
    states = np.arange(1 << N, dtype=np.uint32)
    bits = ((states[:, None] >> np.arange(N, dtype=np.uint32)[None, :]) & 1).astype(np.int8)
    s = (2 * bits - 1).reshape(-1, L, L)  # s[state, y, x], bit b = y*L + x
    E = -(s * np.roll(s, -1, axis=2)).sum(axis=(1, 2), dtype=np.int64) - (s * np.roll(s, -1, axis=1)).sum(
        axis=(1, 2), dtype=np.int64)
    vals, counts = np.unique(E, return_counts=True)
    return {int(v): int(c) for v, c in zip(vals, counts)}, E.astype(np.int32)


def lnZ_from_dos(dos, beta, dps=60):
    mp.dps = dps
    return log(sum(mpf(g) * exp(-mpf(beta) * E) for E, g in dos.items()))
