"""Pins for the CPU oracle (`-m "not gpu"`): every check compares oracle/ with something other
than itself -- the definition Eq. (1) by brute force, closed forms, invariants, textbook routines
(SURVEY.md §8(c) P1-P12).  A plausible mistake anywhere in the oracle (dropped term, wrong sign
or index, transposed operand, off-by-one in a predicate) fails at least one of them."""
from fractions import Fraction
from pathlib import Path

import numpy as np
import pytest

from oracle import oracle as O
from paper_2606_06641_b200 import instances as I
from tests import refmath as R

ALL_TYPES = [R.OR, R.XOR, R.ATLEAST, R.ATMOST, R.EXACTLY, R.NAE]
rng0 = np.random.default_rng(20260641)


def _cases(kmax, kmin=1):
    for k in range(kmin, kmax + 1):
        for t in ALL_TYPES:
            for p in R.all_params(t, k):
                yield t, k, p


# ---------------------------------------------------------------- semantics (O2)
def test_truth_tables_k3_handwritten():
    """Table 1 / Table 2: hand-written k=3 truth tables."""
    for (t, p), sat in R.TRUTH_K3.items():
        g = O.truth_table(t, 3, p)
        assert list(g) == [(-1 if s else 1) for s in sat], (t, p)


def test_truth_tables_all_k():
    for t, k, p in _cases(64, 1):
        if k not in (1, 2, 3, 7, 12, 31, 50, 64):
            continue
        g = O.truth_table(t, k, p)
        want = [(-1 if R.is_sat(t, k, p, tau) else 1) for tau in range(k + 1)]
        assert list(g) == want, (t, k, p)


def test_aliases_and_card_normalisation():
    """AMO = ATMOST 1, EO = EXACTLY 1, OR = ATLEAST 1; CARD '< t' == ATMOST(t-1), '> t' ==
    ATLEAST(t+1), '<= t' == ATMOST(t)."""
    for k in (1, 2, 5, 9):
        assert list(O.truth_table(R.OR, k, 0)) == list(O.truth_table(R.ATLEAST, k, 1))
        amo = [(-1 if tau <= 1 else 1) for tau in range(k + 1)]
        eo = [(-1 if tau == 1 else 1) for tau in range(k + 1)]
        assert list(O.truth_table(R.ATMOST, k, 1)) == amo
        assert list(O.truth_table(R.EXACTLY, k, 1)) == eo
        for t in range(1, k + 1):
            lt = [(-1 if tau < t else 1) for tau in range(k + 1)]
            assert list(O.truth_table(R.ATMOST, k, t - 1)) == lt


# ---------------------------------------------------------------- P1 brute force of Eq. (1)
@pytest.mark.parametrize("k", list(range(1, 11)))
def test_P1_bruteforce_coefficients_and_fe(k):
    for t in ALL_TYPES:
        params = R.all_params(t, k)
        if k >= 9:                       # keep the 4^k work bounded: a spread of parameters
            params = sorted(set([params[0], params[len(params) // 2], params[-1]]))
        for p in params:
            full = R.brute_coeffs(t, k, p)               # 2^k * f^(S) for all 2^k subsets
            A = O.coeffs(t, k, p)
            size = np.array([bin(S).count("1") for S in range(1 << k)])
            assert np.array_equal(full, A[size]), (t, k, p)   # depends on |S| only, == A_|S|
            for trial in range(2):
                y = rng0.uniform(-1, 1, size=k)
                if trial == 1:
                    y[rng0.integers(0, k)] = rng0.choice([-1.0, 1.0])   # a clamped literal
                fe_b, gr_b = R.brute_fe(full, k, y)
                fe_o, gr_o = O.fe_single(t, k, p, y)
                assert abs(fe_o - float(fe_b)) < 1e-14 * (1 + k), (t, k, p)
                assert np.max(np.abs(gr_o - gr_b.astype(np.float64))) < 1e-14 * (1 + k), (t, k, p)


def test_worked_values_k3_golden():
    """tests/golden/worked_k3.txt; each row is first re-derived in exact
    rational arithmetic from Eq. (1), then the oracle must reproduce it exactly (all dyadic)."""
    y = [Fraction(1, 2), Fraction(-1, 4), Fraction(3, 4)]
    yf = np.array([float(v) for v in y])
    rows = [ln for ln in (Path(__file__).parent / "golden" / "worked_k3.txt").read_text().splitlines()
            if ln.strip() and not ln.startswith("#")]
    assert len(rows) == 7
    for ln in rows:
        head, a_s, fe_s, g_s = [s.strip() for s in ln.split("|")]
        _, t, p = head.split()
        t, p = int(t), int(p)
        A_gold = [int(v) for v in a_s.split()]
        fe_gold = float(fe_s)
        g_gold = [float(v) for v in g_s.split()]
        fe_x, g_x = R.brute_fe_exact(t, 3, p, y)
        assert float(fe_x) == fe_gold and [float(v) for v in g_x] == g_gold, head
        assert list(O.coeffs(t, 3, p)) == A_gold, head
        fe_o, g_o = O.fe_single(t, 3, p, yf)
        assert fe_o == fe_gold and list(g_o) == g_gold, head


# ---------------------------------------------------------------- P2 corners
def test_P2_corner_exactness():
    """FE(y) = g(tau) exactly (+-1) at every corner: PAPER.md:57."""
    for t, k, p in _cases(12):
        if k > 8 and p not in (0, 1, k // 2, k):
            continue
        z = R.corners(k) if k <= 8 else R.corners(k)[rng0.integers(0, 1 << k, size=64)]
        for row in z:
            tau = int((row < 0).sum())
            want = -1.0 if R.is_sat(t, k, p, tau) else 1.0
            assert O.fe_single(t, k, p, row.astype(np.float64), grad=False) == want, (t, k, p, tau)


def test_P2_corner_long_constraints():
    for k in (20, 33, 50):
        for t in ALL_TYPES:
            for p in sorted(set([R.all_params(t, k)[0], k // 3, R.all_params(t, k)[-1]])):
                for tau in (0, 1, k // 2, k - 1, k):
                    y = np.ones(k)
                    y[rng0.permutation(k)[:tau]] = -1.0
                    want = -1.0 if R.is_sat(t, k, p, tau) else 1.0
                    got = O.fe_single(t, k, p, y, grad=False)
                    assert abs(got - want) < 1e-12, (t, k, p, tau, got)


# ---------------------------------------------------------------- P3 closed forms
def test_P3_closed_forms_or_xor_nae():
    for k in (1, 2, 3, 5, 7, 8, 13, 20, 40):
        for _ in range(4):
            y = rng0.uniform(-1, 1, size=k).astype(np.longdouble)
            f_or = -1 + 2 * np.prod((1 + y) / 2)          # violated only at the all-false corner
            f_xo = np.prod(y)                             # odd parity: FE = prod y
            f_na = -1 + 2 * (np.prod((1 + y) / 2) + np.prod((1 - y) / 2))
            yd = y.astype(np.float64)
            assert abs(O.fe_single(R.OR, k, 0, yd, grad=False) - float(f_or)) < 1e-14
            assert abs(O.fe_single(R.XOR, k, 1, yd, grad=False) - float(f_xo)) < 1e-14
            assert abs(O.fe_single(R.XOR, k, 0, yd, grad=False) + float(f_xo)) < 1e-14
            assert abs(O.fe_single(R.NAE, k, 0, yd, grad=False) - float(f_na)) < 1e-14


# ---------------------------------------------------------------- P4 Poisson-binomial identity
@pytest.mark.parametrize("k", [1, 2, 3, 6, 11, 17, 24, 33, 41, 50])
def test_P4_expectation_identity(k):
    """FE(y) = E[g(T)], any k, cancellation-free reference."""
    for t in ALL_TYPES:
        params = R.all_params(t, k)
        for p in sorted(set([params[0], params[len(params) // 3], params[len(params) // 2], params[-1]])):
            for mode in ("uniform", "near_corner", "clamped"):
                y = rng0.uniform(-1, 1, size=k)
                if mode == "near_corner":
                    y = np.sign(y) * rng0.uniform(0.9, 1.0, size=k)
                elif mode == "clamped":
                    y[rng0.random(k) < 0.5] = 1.0
                got = O.fe_single(t, k, p, y, grad=False)
                want = float(R.fe_expectation(t, k, p, y))
                assert abs(got - want) < 2e-13, (t, k, p, mode, got, want)
                assert abs(got) <= 1 + 1e-12                                  # P9 range


def test_P4_k64_loose():
    """At k = 64 the long-double ESP sum itself loses digits (terms ~2^32): documented bound."""
    for t in (R.ATLEAST, R.EXACTLY, R.OR):
        y = rng0.uniform(-1, 1, size=64)
        got = O.fe_single(t, 64, 32 if t != R.OR else 0, y, grad=False)
        assert abs(got - float(R.fe_expectation(t, 64, 32 if t != R.OR else 0, y))) < 1e-9


# ---------------------------------------------------------------- P5 / P11 gradient
def test_P5_affine_identity_and_finite_differences():
    for t, k, p in _cases(14):
        if k > 6 and p not in (0, 1, k // 2, k - 1):
            continue
        y = rng0.uniform(-1, 1, size=k)
        fe, g = O.fe_single(t, k, p, y)
        for i in range(k):
            yp, ym = y.copy(), y.copy()
            yp[i], ym[i] = 1.0, -1.0
            exact = (O.fe_single(t, k, p, yp, grad=False) - O.fe_single(t, k, p, ym, grad=False)) / 2
            assert abs(g[i] - exact) < 1e-14, (t, k, p, i)          # FE affine in each coordinate
            h = 1e-4
            yp, ym = y.copy(), y.copy()
            yp[i] += h
            ym[i] -= h
            fd = (O.fe_single(t, k, p, yp, grad=False) - O.fe_single(t, k, p, ym, grad=False)) / (2 * h)
            assert abs(g[i] - fd) < 1e-10, (t, k, p, i)
            assert abs(g[i]) <= 1 + 1e-12                             # P9


@pytest.mark.parametrize("k", [3, 8, 19, 37, 50])
def test_P11_monotone_gradient_closed_form(k):
    """ATLEAST(t): dFE/dy_i = +Pr[T_-i = t-1]; ATMOST(t): -Pr[T_-i = t] (expectation reading)."""
    for tt in sorted(set([1, k // 4, k // 2, k - 1, k])):
        y = rng0.uniform(-1, 1, size=k)
        _, g_al = O.fe_single(R.ATLEAST, k, tt, y)
        _, g_am = O.fe_single(R.ATMOST, k, tt, y)
        for i in rng0.permutation(k)[:5]:
            pm = R.poisson_binomial_pmf((1 - np.delete(y, i)) / 2)
            want_al = float(pm[tt - 1]) if tt >= 1 else 0.0      # ATLEAST(0) is constant
            assert abs(g_al[i] - want_al) < 2e-13
            want_am = -float(pm[tt]) if tt <= k - 1 else 0.0
            assert abs(g_am[i] - want_am) < 2e-13
        assert (g_al >= -1e-15).all() and (g_am <= 1e-15).all()
    _, g_or = O.fe_single(R.OR, k, 0, rng0.uniform(-1, 1, size=k))
    assert (g_or >= 0).all()


# ---------------------------------------------------------------- P6 / P7 coefficients
def test_P6_parseval_and_P7_mean_exact():
    from math import comb
    for t, k, p in _cases(62):
        if k > 12 and (k % 7 or p not in (0, 1, k // 2, k)):
            continue
        A = [int(a) for a in O.coeffs(t, k, p)]
        assert sum(comb(k, j) * A[j] * A[j] for j in range(k + 1)) == 4 ** k, (t, k, p)
        n_sat = sum(comb(k, tau) for tau in range(k + 1) if R.is_sat(t, k, p, tau))
        assert A[0] == 2 ** k - 2 * n_sat, (t, k, p)


# ---------------------------------------------------------------- P8 dualities
def test_P8_dualities():
    for k in (1, 2, 4, 7, 12, 25):
        y = rng0.uniform(-1, 1, size=k)
        fe = lambda t, p, yy=y: O.fe_single(t, k, p, yy, grad=False)
        for tt in range(0, k + 1):
            assert abs(fe(R.ATMOST, tt) - fe(R.ATLEAST, k - tt, -y)) < 1e-14
            nxt = fe(R.ATLEAST, tt + 1) if tt + 1 <= k else 1.0
            assert abs(fe(R.EXACTLY, tt) - (1 + fe(R.ATLEAST, tt) - nxt)) < 1e-14
            assert abs(fe(R.ATMOST, tt) + nxt) < 1e-14
        assert abs(fe(R.NAE, 0) - fe(R.NAE, 0, -y)) < 1e-15
        assert abs(fe(R.XOR, 1, -y) - (-1) ** k * fe(R.XOR, 1)) < 1e-15
        assert abs(fe(R.OR, 0) - fe(R.ATLEAST, 1)) < 1e-15
        # even-parity XOR == odd-parity XOR with one literal's sign flipped (reading A13)
        y2 = y.copy()
        y2[0] = -y2[0]
        assert abs(fe(R.XOR, 0) - fe(R.XOR, 1, y2)) < 1e-15


# ---------------------------------------------------------------- instance level (O1, O4, O7, O8)
def _small_instance(seed, with_fixed):
    return I.make_mixed(n=14, m=40, kmin=1, kmax=9, seed=seed, batch=5, with_fixed=with_fixed)


@pytest.mark.parametrize("with_fixed", [False, True])
def test_instance_eval_grad_against_bruteforce_composition(with_fixed):
    inst = _small_instance(11, with_fixed)
    B = 5
    X = I.make_x0(inst, seed=3, batch=B, dtype=np.float64)
    X[2, 0], X[3, 1], X[4, 2] = 1.0, -1.0, 0.0
    if with_fixed:
        fx = inst.fixed != 0
        X[fx, :B] = 0.37          # whatever X holds, fixed variables use their fixed value (A17)
    F, G = O.eval_grad(inst, X, B)
    Fw = np.zeros(B, dtype=np.longdouble)
    Gw = np.zeros((inst.n_vars, B), dtype=np.longdouble)
    for b in range(B):
        xb = X[:, b].copy()
        if with_fixed:
            xb[fx] = inst.fixed[fx]
        for c in range(inst.n_cons):
            lo, hi = int(inst.row_ptr[c]), int(inst.row_ptr[c + 1])
            v, s = inst.lit_var[lo:hi], inst.lit_sign[lo:hi].astype(np.float64)
            full = R.brute_coeffs(int(inst.ctype[c]), hi - lo, int(inst.param[c]))
            fe, gr = R.brute_fe(full, hi - lo, s * xb[v])
            Fw[b] += fe
            Gw[v, b] += s * gr
    if with_fixed:
        Gw[fx, :] = 0
        assert np.all(G[fx, :B] == 0.0)                    # gradient masking
    assert np.max(np.abs(F - Fw.astype(np.float64))) < 1e-12
    assert np.max(np.abs(G[:, :B] - Gw.astype(np.float64))) < 1e-12
    assert np.all(G[:, B:] == 0.0)


def test_sum_is_minus_m_iff_satisfied():
    """X satisfies phi iff sum_k FE = -m (on corners)."""
    base = I.make_mixed(n=30, m=60, kmin=1, kmax=10, seed=5, batch=8)
    base.meta["admissible"] = [R.admissible_taus(int(t), int(k), int(p)) or [0]
                               for t, k, p in zip(base.ctype, base.lengths(), base.param)]
    keep = [c for c in range(base.n_cons) if R.admissible_taus(int(base.ctype[c]),
            int(base.lengths()[c]), int(base.param[c]))]
    assert len(keep) > 40
    inst, hidden = I.plant_solution(base, seed=2)
    B = 8
    T = np.repeat(hidden[:, None], B, axis=1)
    for b in range(1, B):
        T[rng0.integers(0, inst.n_vars, size=b), b] ^= True
    X = I.corner_x(inst, T, dtype=np.float64)
    F = O.eval_grad(inst, X, B, grad=False)
    sat, sol = O.check(inst, X, B)
    unsat_possible = inst.n_cons - len(keep)           # constraints with no satisfying count
    assert sat[0] == inst.n_cons - unsat_possible
    # F = (#violated) - (#satisfied) exactly on corners
    assert np.array_equal(F, (inst.n_cons - sat) - sat.astype(np.float64))
    assert np.array_equal(sol, (sat == inst.n_cons).astype(np.uint8))


# ---------------------------------------------------------------- P12 discrete check (O10)
@pytest.mark.parametrize("with_fixed", [False, True])
def test_P12_check_against_independent_recount(with_fixed):
    inst = I.make_mixed(n=40, m=120, kmin=1, kmax=16, seed=21, batch=16, with_fixed=with_fixed)
    B = 16
    X = I.make_x0(inst, seed=8, batch=B, dtype=np.float64)
    X[0, :] = 0.0           # tie: rounds to False (reading A9)
    X[1, :] = -0.0          # IEEE -0.0 < 0 is false -> False
    X[2, :] = 1.0
    X[3, :] = -1.0
    X[4, :] = -1e-300
    X[5, :] = 5e-324
    if with_fixed:
        fx = inst.fixed != 0
        X[fx, :B] = -X[fx, :B] * 0.5      # garbage in fixed rows must be ignored
    sat, sol = O.check(inst, X, B)
    want = R.recount(inst, X, B)
    assert np.array_equal(sat, want)
    assert np.array_equal(sol, (want == inst.n_cons).astype(np.uint8))


def test_P12_planted_solution_and_single_flip():
    base = I.make_config(2, scale=0.02, batch=4)
    base.meta["admissible"] = [R.admissible_taus(int(t), int(k), int(p))
                               for t, k, p in zip(base.ctype, base.lengths(), base.param)]
    inst, hidden = I.plant_solution(base, seed=4)
    B = 4
    T = np.repeat(hidden[:, None], B, axis=1)
    free = np.nonzero(inst.fixed == 0)[0]
    for b in range(1, B):
        T[free[rng0.integers(0, free.size)], b] ^= True
    X = I.corner_x(inst, T, dtype=np.float64) * 0.25       # off-corner magnitudes, same signs
    sat, sol = O.check(inst, X, B)
    assert sat[0] == inst.n_cons and sol[0] == 1
    assert np.array_equal(sat, R.recount(inst, X, B))
    assert np.array_equal(sol, (sat == inst.n_cons).astype(np.uint8))


# ---------------------------------------------------------------- O9 + freeze: the step loop
@pytest.mark.parametrize("with_fixed", [False, True])
def test_step_composition_and_freeze(with_fixed):
    """oracle.step == gradient at X(t-1) -> clamp(x - eta g) on free vars -> check X(t) -> freeze;
    recomposed here from eval_grad/check + numpy (Alg. 1)."""
    base = I.make_mixed(n=24, m=30, kmin=2, kmax=4, seed=31, batch=24, with_fixed=with_fixed,
                        types=[R.OR, R.XOR, R.NAE])
    base.meta["admissible"] = [R.admissible_taus(int(t), int(k), int(p))
                               for t, k, p in zip(base.ctype, base.lengths(), base.param)]
    inst, _ = I.plant_solution(base, seed=9)
    B, eta, T = 24, 0.25, 30
    X0 = I.make_x0(inst, seed=12, batch=B, dtype=np.float64)
    Xo, Fo, sato, solo, firsto = O.step(inst, X0, eta, T, B)
    X = X0.copy()
    sol = np.zeros(B, dtype=bool)
    first = np.full(B, -1)
    free = np.ones(inst.n_vars, dtype=bool) if inst.fixed is None else (inst.fixed == 0)
    for t in range(1, T + 1):
        _, G = O.eval_grad(inst, X, B)
        Xn = np.clip(X.astype(np.longdouble) - np.longdouble(eta) * G.astype(np.longdouble), -1, 1)
        upd = free[:, None] & ~sol[None, :]
        X[:, :B] = np.where(upd, Xn[:, :B].astype(np.float64), X[:, :B])
        sat, _ = O.check(inst, X, B)
        newly = (sat == inst.n_cons) & ~sol
        first[newly] = t
        sol |= newly
    assert sol.sum() >= 1 and (~sol).sum() >= 1, "test should exercise both solved and unsolved"
    assert np.array_equal(solo.astype(bool), sol)
    assert np.array_equal(firsto, first)
    assert np.max(np.abs(Xo - X)) < 1e-13
    assert np.array_equal(sato, O.check(inst, Xo, B)[0])
    assert np.max(np.abs(Fo - O.eval_grad(inst, Xo, B, grad=False))) < 1e-12
    assert np.all(np.abs(Xo[:, :B]) <= 1.0)
    # resume: 30 steps == 10 steps + 20 resumed steps
    Xa, _, _, sola, firsta = O.step(inst, X0, eta, 10, B)
    Xb, _, satb, solb, firstb = O.step(inst, Xa, eta, 20, B, step_base=10, state=(sola, firsta))
    assert np.array_equal(Xb, Xo) and np.array_equal(solb, solo) and np.array_equal(firstb, firsto)


# ---------------------------------------------------------------- O11: Alg. 1 with line search (reading B5)
def _ls_recompose(inst, X0, B, T, s_max, beta, c1, delta, J):
    """oracle.step_ls recomposed from eval_grad / check and numpy long doubles."""
    X = X0.copy()
    sol = np.zeros(B, dtype=bool); conv = np.zeros(B, dtype=bool)
    first = np.full(B, -1); eta_last = np.full(B, s_max, dtype=np.longdouble)
    free = np.ones(inst.n_vars, dtype=bool) if inst.fixed is None else (inst.fixed == 0)
    accepted_etas = [[] for _ in range(B)]
    for t in range(1, T + 1):
        F0, G = O.eval_grad(inst, X, B)
        for b in range(B):
            if sol[b] or conv[b]:
                continue
            eta = np.longdouble(s_max)
            x0 = X[:, b].astype(np.longdouble); g = G[:, b].astype(np.longdouble)
            for _ in range(J):
                xt = np.where(free, np.clip(x0 - eta * g, -1, 1), x0)
                D = np.sum(g * (x0 - xt))
                Xt = X[:, b:b + 1].copy(); Xt[:, 0] = xt.astype(np.float64)
                F1 = O.eval_grad(inst, np.ascontiguousarray(Xt), 1, grad=False)[0]
                if F1 <= F0[b] - c1 * D:
                    X[:, b] = xt.astype(np.float64); accepted_etas[b].append(float(eta))
                    break
                eta = eta * beta
                if eta < delta:
                    conv[b] = True
                    break
            eta_last[b] = eta
        sat, _ = O.check(inst, X, B)
        newly = (sat == inst.n_cons) & ~sol & ~conv
        # a candidate that converged in this very step is still checked (Alg. 1 checks X(t) every step)
        newly |= (sat == inst.n_cons) & ~sol
        first[newly] = t
        sol |= newly
    return X, sol, conv, first, eta_last, accepted_etas


@pytest.mark.parametrize("with_fixed", [False, True])
def test_step_ls_composition(with_fixed):
    """oracle.step_ls == Alg. 1 with backtracking (reading B5) recomposed from eval_grad / check."""
    base = I.make_mixed(n=20, m=26, kmin=2, kmax=4, seed=41, batch=12, with_fixed=with_fixed,
                        types=[R.OR, R.XOR, R.NAE])
    base.meta["admissible"] = [R.admissible_taus(int(t), int(k), int(p))
                               for t, k, p in zip(base.ctype, base.lengths(), base.param)]
    inst, _ = I.plant_solution(base, seed=5)
    B, T = 12, 12
    kw = dict(s_max=2.0, beta=0.5, c1=1e-4, delta=1e-3, max_trials=6)
    X0 = I.make_x0(inst, seed=3, batch=B, dtype=np.float64)
    Xo, Fo, etao, sato, solo, firsto, convo, margin = O.step_ls(inst, X0, T, B, **kw)
    X, sol, conv, first, eta_last, _ = _ls_recompose(inst, X0, B, T, kw["s_max"], kw["beta"], kw["c1"], kw["delta"],
                                                     kw["max_trials"])
    assert np.array_equal(solo.astype(bool), sol) and np.array_equal(firsto, first)
    assert np.array_equal(convo.astype(bool), conv)
    assert np.max(np.abs(Xo - X)) < 1e-13
    assert np.array_equal(sato, O.check(inst, Xo, B)[0])
    assert np.max(np.abs(Fo - O.eval_grad(inst, Xo, B, grad=False))) < 1e-12
    assert np.all(np.abs(Xo[:, :B]) <= 1.0)
    # resume: T steps == 5 steps + (T - 5) resumed steps
    Xa, _, _, _, sola, firsta, conva, _ = O.step_ls(inst, X0, 5, B, **kw)
    Xb, _, _, _, solb, firstb, convb, _ = O.step_ls(inst, Xa, T - 5, B, step_base=5, state=(sola, firsta, conva), **kw)
    assert np.array_equal(Xb, Xo) and np.array_equal(solb, solo) and np.array_equal(firstb, firsto)
    assert np.array_equal(convb, convo)


def test_step_ls_textbook_properties():
    """What the Armijo rule along the projection arc guarantees, whatever the constants:
    F never increases, every accepted step satisfies the sufficient-decrease inequality, eta is on the
    ladder s_max beta^j, a huge delta freezes everything at once, and with beta-ladder exhausted (one
    trial, absurd s_max) X stays put when the single trial is rejected."""
    inst = I.make_mixed(n=30, m=60, kmin=2, kmax=6, seed=77, batch=16, types=[R.OR, R.XOR, R.ATLEAST, R.NAE])
    B = 16
    X0 = I.make_x0(inst, seed=8, batch=B, dtype=np.float64)
    F_prev = O.eval_grad(inst, X0, B, grad=False)
    X = X0
    state = None
    for t in range(6):
        Xn, F, eta, sat, sol, first, conv, margin = O.step_ls(inst, X, 1, B, s_max=4.0, beta=0.5, c1=1e-3, delta=1e-9,
                                                              max_trials=40, step_base=t, state=state)
        assert np.all(F <= F_prev + 1e-15)                            # monotone descent
        ladder = np.log2(4.0 / eta)
        assert np.all(np.abs(ladder - np.round(ladder)) < 1e-12) and np.all(eta <= 4.0)
        moved = np.any(Xn != X, axis=0)[:B]
        _, G = O.eval_grad(inst, X, B)
        D = np.sum(G[:, :B] * (X[:, :B] - Xn[:, :B]), axis=0)
        assert np.all(F[moved] <= F_prev[moved] - 1e-3 * D[moved] + 1e-15)   # sufficient decrease where it moved
        assert np.all(D[moved] >= 0)
        X, F_prev, state = Xn, F, (sol, first, conv)
    # delta above s_max * beta: the first rejection converges the candidate; accepted ones still move
    Xn, F, eta, sat, sol, first, conv, _ = O.step_ls(inst, X0, 3, B, s_max=64.0, beta=0.5, c1=0.5, delta=40.0, max_trials=5)
    assert np.all(conv[np.all(Xn == X0, axis=0)[:B] & (sol == 0)] == 1)
    assert np.all(np.abs(Xn) <= 1.0)
    with pytest.raises(ValueError):
        O.step_ls(inst, X0, 1, B, beta=1.5)


# ---------------------------------------------------------------- O12: restart initialisation
def test_restart_generator_properties():
    """The generator is fixed by include/afsat.h; what pins it here: one value worked out by hand-coded
    integer arithmetic in Python, range [-1, 1) on the 2^-23 grid, uniformity (chi-square), independence of
    seed / round / candidate / variable streams, fixed variables and kept candidates."""
    inst = I.make_mixed(n=64, m=10, kmin=2, kmax=4, seed=3, batch=256, with_fixed=True)
    B = 256
    X0 = np.zeros((64, 256))
    Xa = O.restart(inst, X0, seed=0x123456789ABCDEF, round_=3, B=B)
    # the formula, retyped with Python integers for one (b, v)
    M = 0xFFFFFFFF
    def fmix(h):
        h ^= h >> 16; h = (h * 0x85EBCA6B) & M; h ^= h >> 13; h = (h * 0xC2B2AE35) & M; h ^= h >> 16
        return h
    free = np.nonzero(inst.fixed == 0)[0]
    v, b = int(free[5]), 77
    lo, hi = 0x123456789ABCDEF & M, 0x123456789ABCDEF >> 32
    h = fmix((fmix(((fmix(lo ^ ((b * 0x9E3779B9) & M)) + v * 0x85EBCA6B) & M) ^ hi) + 3 * 0xC2B2AE35) & M)
    assert Xa[v, b] == (h >> 8) / 2.0 ** 23 - 1.0
    vals = Xa[free][:, :B].ravel()
    assert vals.min() >= -1.0 and vals.max() < 1.0
    assert np.all(vals * 2 ** 23 == np.round(vals * 2 ** 23))         # on the fp32-exact grid
    hist, _ = np.histogram(vals, bins=32, range=(-1, 1))
    exp = vals.size / 32
    assert np.sum((hist - exp) ** 2 / exp) < 80                       # chi-square, 31 dof (p ~ 1e-6 at 80)
    assert abs(vals.mean()) < 0.02
    fx = inst.fixed != 0
    assert np.all(Xa[fx][:, :B] == inst.fixed[fx][:, None])           # fixed variables hold their value
    for other in (O.restart(inst, X0, seed=0x123456789ABCDEF, round_=4, B=B),
                  O.restart(inst, X0, seed=0x123456789ABCDEE, round_=3, B=B),
                  O.restart(inst, X0, seed=0x023456789ABCDEF, round_=3, B=B)):
        assert abs(np.corrcoef(other[free][:, :B].ravel(), vals)[0, 1]) < 0.04   # ~4.5 sigma at 13 000 samples
    assert abs(np.corrcoef(Xa[free][:, 0], Xa[free][:, 1])[0, 1]) < 0.5
    assert abs(np.corrcoef(Xa[free[0], :B], Xa[free[1], :B])[0, 1]) < 0.2
    keep = (np.arange(B) % 3 == 0).astype(np.uint8)
    Xk = O.restart(inst, X0 + 0.25, seed=7, round_=0, B=B, keep=keep)
    assert np.all(Xk[:, :B][:, keep != 0] == 0.25)
    assert np.array_equal(Xk[:, :B][:, keep == 0], O.restart(inst, X0, seed=7, round_=0, B=B)[:, :B][:, keep == 0])


def test_rejects_bad_input():
    inst = I.make_mixed(n=10, m=5, kmin=2, kmax=4, seed=1, batch=2)
    X = I.make_x0(inst, batch=2, dtype=np.float64)
    bad = I.Instance(**{**inst.__dict__})
    bad.lit_var = inst.lit_var.copy()
    bad.lit_var[1] = bad.lit_var[0]          # repeated variable inside one constraint (A15)
    with pytest.raises(ValueError):
        O.eval_grad(bad, X, 2)
    bad.lit_var = inst.lit_var.copy()
    bad.lit_sign = inst.lit_sign.copy()
    bad.lit_sign[0] = 0
    with pytest.raises(ValueError):
        O.check(bad, X, 2)
