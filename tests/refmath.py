"""Independent mathematics used to PIN the oracle (and, for the host tables, the CUDA library).

Nothing here is imported by oracle/ or by the product package, and nothing here imports them.
Each routine is a definition or a textbook routine that the paper's quantities must agree with:

  * ``TRUTH_K3`` / ``is_sat``: the constraint semantics written out from the PB forms of
    PAPER.md Table 1 (:87-97) and Table 2 (:252-262, :264).
  * ``brute_coeffs`` / ``brute_fe``: Eq. (1) expanded over all 2^k subsets with
    f^(S) = 2^-k sum_z f(z) prod_{i in S} z_i over all 2^k corners (definition of the
    Walsh-Fourier coefficients, the paper's ref. [6]).
  * ``poisson_binomial_pmf``: the standard DP for the number of successes of independent
    Bernoulli trials; FE(y) = E[g(T)] with p_i = (1 - y_i)/2 because a multilinear polynomial
    evaluated at means equals the expectation over independent +-1 coordinates.
"""
from __future__ import annotations

from fractions import Fraction

import numpy as np

OR, XOR, ATLEAST, ATMOST, EXACTLY, NAE = 0, 1, 2, 3, 4, 5

# Hand-written truth tables for k = 3: index tau = number of true literals, value True = satisfied.
TRUTH_K3 = {
    (OR, 0): [False, True, True, True],          # sum >= 1
    (XOR, 1): [False, True, False, True],        # sum odd  (the paper's XOR)
    (XOR, 0): [True, False, True, False],        # sum even
    (NAE, 0): [False, True, True, False],        # not all equal
    (ATLEAST, 2): [False, False, True, True],    # sum >= 2
    (ATMOST, 1): [True, True, False, False],     # sum <= 1 (AMO)
    (EXACTLY, 1): [False, True, False, False],   # sum == 1 (EO)
    (EXACTLY, 2): [False, False, True, False],
    (ATLEAST, 0): [True, True, True, True],
    (ATMOST, 3): [True, True, True, True],
    (ATMOST, 0): [True, False, False, False],
    (ATLEAST, 3): [False, False, False, True],
}


def is_sat(ctype: int, k: int, param: int, tau: int) -> bool:
    """Table 1 / Table 2 semantics as set membership of tau (written independently of the
    oracle's switch: each type lists the admissible counts)."""
    admissible = {
        OR: set(range(1, k + 1)),
        XOR: {t for t in range(k + 1) if t % 2 == param % 2},
        ATLEAST: {t for t in range(k + 1) if t >= param},
        ATMOST: {t for t in range(k + 1) if t <= param},
        EXACTLY: {param} & set(range(k + 1)),
        NAE: set(range(1, k)),
    }[ctype]
    return tau in admissible


def admissible_taus(ctype: int, k: int, param: int):
    return [t for t in range(k + 1) if is_sat(ctype, k, param, t)]


def all_params(ctype: int, k: int):
    if ctype in (OR, NAE):
        return [0]
    if ctype == XOR:
        return [0, 1]
    return list(range(0, k + 1))


def corners(k: int) -> np.ndarray:
    """All 2^k corners z in {+1,-1}^k, row r has z_i = -1 iff bit i of r is set."""
    r = np.arange(1 << k)[:, None]
    return np.where((r >> np.arange(k)[None, :]) & 1, -1, 1).astype(np.int64)


def brute_coeffs(ctype: int, k: int, param: int) -> np.ndarray:
    """2^k * f^(S) for every subset S (index = bitmask), exact int64, straight from the
    definition: sum over ALL corners of f(z) * prod_{i in S} z_i."""
    z = corners(k)                                        # [2^k, k]
    tau = (z < 0).sum(axis=1)
    f = np.array([-1 if is_sat(ctype, k, param, int(t)) else 1 for t in tau], dtype=np.int64)
    masks = np.arange(1 << k)
    # chi_S(z) = (-1)^{|S ∩ {i: z_i=-1}|}; corner index r IS the bitmask of -1 entries
    inter = masks[:, None] & masks[None, :]
    pop = np.zeros_like(inter)
    for b in range(k):
        pop += (inter >> b) & 1
    chi = 1 - 2 * (pop & 1)                               # [S, z]
    return chi @ f                                        # exact integers


def brute_fe(coef_scaled: np.ndarray, k: int, y: np.ndarray):
    """FE(y) = sum_S f^(S) prod_{i in S} y_i and its gradient, all 2^k terms, in long double."""
    y = np.asarray(y, dtype=np.longdouble)
    masks = np.arange(1 << k)
    bits = ((masks[:, None] >> np.arange(k)[None, :]) & 1).astype(bool)   # [S, i]
    mono = np.prod(np.where(bits, y[None, :], np.longdouble(1)), axis=1)
    scale = np.longdouble(2) ** (-k)
    fe = (coef_scaled.astype(np.longdouble) * mono).sum() * scale
    grad = np.zeros(k, dtype=np.longdouble)
    for i in range(k):
        others = bits.copy()
        others[:, i] = False
        mono_i = np.prod(np.where(others, y[None, :], np.longdouble(1)), axis=1)
        grad[i] = (coef_scaled.astype(np.longdouble) * mono_i * bits[:, i]).sum() * scale
    return fe, grad


def brute_fe_exact(ctype, k, param, y_frac):
    """Same as brute_fe in exact rational arithmetic (tiny k only)."""
    coef = brute_coeffs(ctype, k, param)
    fe = Fraction(0)
    grad = [Fraction(0)] * k
    for S in range(1 << k):
        mono = Fraction(1)
        for i in range(k):
            if S >> i & 1:
                mono *= y_frac[i]
        fe += Fraction(int(coef[S]), 1 << k) * mono
        for i in range(k):
            if S >> i & 1:
                m = Fraction(1)
                for j in range(k):
                    if j != i and (S >> j & 1):
                        m *= y_frac[j]
                grad[i] += Fraction(int(coef[S]), 1 << k) * m
    return fe, grad


def poisson_binomial_pmf(p) -> np.ndarray:
    """pmf[t] = Pr[T = t], T = sum of independent Bernoulli(p_i); non-negative terms only."""
    p = np.asarray(p, dtype=np.longdouble)
    pmf = np.zeros(p.shape[0] + 1, dtype=np.longdouble)
    pmf[0] = 1
    for i, pi in enumerate(p):
        pmf[1:i + 2] = pmf[1:i + 2] * (1 - pi) + pmf[0:i + 1] * pi
        pmf[0] = pmf[0] * (1 - pi)
    return pmf


def fe_expectation(ctype, k, param, y):
    """FE(y) = sum_tau g(tau) Pr[T = tau] with literal i true with probability (1 - y_i)/2."""
    y = np.asarray(y, dtype=np.longdouble)
    pmf = poisson_binomial_pmf((1 - y) / 2)
    g = np.array([-1 if is_sat(ctype, k, param, t) else 1 for t in range(k + 1)],
                 dtype=np.longdouble)
    return (g * pmf).sum()


def recount(inst, X, B):
    """Independent integer recount of satisfied constraints (plain loops)."""
    sat = np.zeros(B, dtype=np.int64)
    for b in range(B):
        for c in range(inst.n_cons):
            lo, hi = int(inst.row_ptr[c]), int(inst.row_ptr[c + 1])
            tau = 0
            for p in range(lo, hi):
                v = int(inst.lit_var[p])
                if inst.fixed is not None and inst.fixed[v] != 0:
                    var_true = inst.fixed[v] < 0
                else:
                    var_true = bool(X[v, b] < 0)
                tau += int(var_true if inst.lit_sign[p] > 0 else not var_true)
            sat[b] += int(is_sat(int(inst.ctype[c]), hi - lo, int(inst.param[c]), tau))
    return sat
