"""Exact density of states g(E) of the L x L periodic square-lattice Ising model.

Test infrastructure used ONLY to pin the CPU oracle (it is the paper's own
ground truth: "available analytic solutions for the density of
states [43]", Fig. 7).  The formula is not printed in
PAPER.md; it is Kaufman's finite-torus partition function in the product form
Beale used ([43]), restated in DESIGN.md "Exact density of states":

  x = exp(-2K),  x^N Z(K) = sum_j g(E_j) x^(2j),  E_j = -2N + 4j,  N = L*L, n = m = L even
  A  = (1+x^2)^2 / (x (1-x^2)),   c_l = A - 2 cos(pi l / n),  l = 0..2n-1
  D_0 = 2, D_1 = y, D_{k+1} = y D_k - D_{k-1}                  (D_k(2 cosh g) = 2 cosh k g)
  F_l = D_{m/2}(c_l)
  Z1 = prod_{l odd} F_l          Z2 = prod_{l odd, l<n} (F_l^2 - 4)
  Z3 = prod_{l even} F_l         Z4 = (e0^{m/2} - e0^{-m/2}) (en^{m/2} - en^{-m/2}) prod_{l even, 0<l<n} (F_l^2 - 4)
       e0 = (1-x)/(x(1+x)),  en = (1+x)/(x(1-x))
  x^N Z = x^N ((1-x^2)/x)^{N/2} (Z1 + Z2 + Z3 + Z4) / 2

The polynomial Q(y) = sum_j g_j y^j (y = x^2) is sampled at N+1 points on a
circle of radius 1/2 and recovered by an inverse DFT in arbitrary precision
(mpmath); the result is rounded to integers and self-checked:
sum g = 2^N, g symmetric, g_0 = 2, g_1 = 0, g_2 = 2N, g_3 = 4N, rounding residue tiny.
Independent cross-check for L = 4: brute-force enumeration (tests/test_oracle_pins.py).
"""
import mpmath as mp


def _D(k, y):
    d0, d1 = mp.mpf(2), y
    if k == 0:
        return d0
    for _ in range(k - 1):
        d0, d1 = d1, y * d1 - d0
    return d1


def _xNZ(x, L):
    n = m = L
    N = L * L
    A = (1 + x * x) ** 2 / (x * (1 - x * x))
    F = [_D(m // 2, A - 2 * mp.cos(mp.pi * l / n)) for l in range(2 * n)]
    Z1 = mp.mpf(1)
    Z2 = mp.mpf(1)
    Z3 = mp.mpf(1)
    Z4 = mp.mpf(1)
    for l in range(2 * n):
        if l % 2 == 1:
            Z1 *= F[l]
            if l < n:
                Z2 *= F[l] ** 2 - 4
        else:
            Z3 *= F[l]
            if 0 < l < n:
                Z4 *= F[l] ** 2 - 4
    e0 = (1 - x) / (x * (1 + x))
    en = (1 + x) / (x * (1 - x))
    h = m // 2
    Z4 *= (e0 ** h - e0 ** (-h)) * (en ** h - en ** (-h))
    pref = x ** N * ((1 - x * x) / x) ** (N // 2)
    return pref * (Z1 + Z2 + Z3 + Z4) / 2


def exact_g(L: int, digits: int | None = None):
    """List of N+1 python ints g[j] = number of states with E = -2N + 4j."""
    assert L >= 2 and L % 2 == 0
    N = L * L
    if digits is None:
        digits = max(60, int(0.75 * N) + 40)  # 2^N has 0.30 N digits; radius 1/2 costs another 0.30 N
    with mp.workdps(digits):
        M = N + 1
        rad = mp.mpf(1) / 2
        samples = []
        for k in range(M):
            y = rad * mp.expjpi(mp.mpf(2 * k) / M)
            x = mp.sqrt(y)
            samples.append(_xNZ(x, L))
        g = []
        worst = mp.mpf(0)
        roots = [mp.expjpi(-mp.mpf(2 * k) / M) for k in range(M)]   # exp(-2 pi i k / M), evaluated once (L = 32: minutes -> seconds)
        for j in range(M):
            acc = mp.mpc(0)
            for k in range(M):
                acc += samples[k] * roots[(k * j) % M]
            val = acc / M / rad ** j
            r = mp.nint(val.real)
            worst = max(worst, abs(val.real - r), abs(val.imag))
            g.append(int(r))
        assert worst < mp.mpf(10) ** (-8), f"rounding residue too large: {worst}"
    assert sum(g) == 2 ** N, "sum g != 2^N"
    assert g == g[::-1], "g not symmetric"
    assert g[0] == 2 and g[1] == 0 and g[2] == 2 * N and g[3] == 4 * N
    return g


def ln_g(L: int):
    """float64 list ln g[j]; -inf where g = 0."""
    import math
    out = []
    for v in exact_g(L):
        out.append(float(mp.log(v)) if v > 0 else -math.inf)
    return out
