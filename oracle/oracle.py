"""ctypes wrapper around oracle/afsat_oracle.c -- TEST INFRASTRUCTURE ONLY.

The oracle is the plain long-double CPU implementation of the AFSAT hot path written from the
paper (see the header of afsat_oracle.c for the step-by-step citations).  Only tests/,
__graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this
module; the product package never does, and this module never imports the product package.

Arrays are numpy; X and G are variable-major ``[n, ldb]`` float64.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "afsat_oracle.c"
_LIB = _HERE / "liboracle_afsat.so"
_lib = None


def build(force: bool = False) -> Path:
    """Compile the oracle with gcc (-O2, no fast-math, OpenMP over candidates)."""
    if force or not _LIB.exists() or _LIB.stat().st_mtime < _SRC.stat().st_mtime:
        tmp = _LIB.with_suffix(f".so.tmp{os.getpid()}")
        subprocess.check_call(["gcc", "-O2", "-std=c11", "-fPIC", "-shared", "-fopenmp",
                               "-Wall", "-o", str(tmp), str(_SRC), "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


def _p(a, t):
    return a.ctypes.data_as(C.POINTER(t)) if a is not None else None


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(str(_LIB))
        L.oracle_num_threads.restype = C.c_int
        for name in ("oracle_truth_table", "oracle_coeffs", "oracle_fe_single",
                     "oracle_eval_grad", "oracle_check", "oracle_step", "oracle_step_ls", "oracle_restart"):
            getattr(L, name).restype = C.c_int
        _lib = L
    return _lib


def num_threads() -> int:
    return int(lib().oracle_num_threads())


def truth_table(ctype: int, k: int, param: int) -> np.ndarray:
    g = np.zeros(k + 1, dtype=np.int8)
    rc = lib().oracle_truth_table(C.c_int(ctype), C.c_int(k), C.c_int(param), _p(g, C.c_int8))
    if rc:
        raise ValueError(f"oracle_truth_table rc={rc}")
    return g


def coeffs(ctype: int, k: int, param: int) -> np.ndarray:
    """Exact integers A_j = 2^k * f^(S), |S| = j (k <= 62)."""
    A = np.zeros(k + 1, dtype=np.int64)
    rc = lib().oracle_coeffs(C.c_int(ctype), C.c_int(k), C.c_int(param), _p(A, C.c_int64))
    if rc:
        raise ValueError(f"oracle_coeffs rc={rc}")
    return A


def fe_single(ctype: int, k: int, param: int, y, grad: bool = True):
    """FE and dFE/dy of one constraint at literal values y (length k)."""
    y = np.ascontiguousarray(y, dtype=np.float64)
    assert y.shape == (k,)
    fe = C.c_double(0.0)
    d = np.zeros(k, dtype=np.float64) if grad else None
    rc = lib().oracle_fe_single(C.c_int(ctype), C.c_int(k), C.c_int(param), _p(y, C.c_double),
                                C.byref(fe), _p(d, C.c_double))
    if rc:
        raise ValueError(f"oracle_fe_single rc={rc}")
    return (fe.value, d) if grad else fe.value


def _inst_args(inst):
    row_ptr = np.ascontiguousarray(inst.row_ptr, dtype=np.int64)
    lit_var = np.ascontiguousarray(inst.lit_var, dtype=np.int32)
    lit_sign = np.ascontiguousarray(inst.lit_sign, dtype=np.int8)
    ctype = np.ascontiguousarray(inst.ctype, dtype=np.uint8)
    param = np.ascontiguousarray(inst.param, dtype=np.int32)
    fixed = None if inst.fixed is None else np.ascontiguousarray(inst.fixed, dtype=np.int8)
    keep = (row_ptr, lit_var, lit_sign, ctype, param, fixed)
    args = (C.c_int32(inst.n_vars), C.c_int32(row_ptr.shape[0] - 1), _p(row_ptr, C.c_int64),
            _p(lit_var, C.c_int32), _p(lit_sign, C.c_int8), _p(ctype, C.c_uint8),
            _p(param, C.c_int32), _p(fixed, C.c_int8))
    return args, keep


def _check_x(inst, X, B):
    X = np.ascontiguousarray(X, dtype=np.float64)
    assert X.ndim == 2 and X.shape[0] == inst.n_vars and X.shape[1] >= B
    return X


def eval_grad(inst, X, B=None, grad: bool = True):
    """F[b] = sum_C FE_C(X[:, b]) and G[v, b] (zero rows for fixed variables)."""
    B = int(X.shape[1] if B is None else B)
    X = _check_x(inst, X, B)
    F = np.zeros(B, dtype=np.float64)
    G = np.zeros_like(X) if grad else None
    args, keep = _inst_args(inst)
    rc = lib().oracle_eval_grad(*args, C.c_int32(B), C.c_int64(X.shape[1]), _p(X, C.c_double),
                                _p(F, C.c_double), _p(G, C.c_double))
    if rc:
        raise ValueError(f"oracle_eval_grad rc={rc}")
    return (F, G) if grad else F


def check(inst, X, B=None):
    B = int(X.shape[1] if B is None else B)
    X = _check_x(inst, X, B)
    sat = np.zeros(B, dtype=np.int32)
    sol = np.zeros(B, dtype=np.uint8)
    args, keep = _inst_args(inst)
    rc = lib().oracle_check(*args, C.c_int32(B), C.c_int64(X.shape[1]), _p(X, C.c_double),
                            _p(sat, C.c_int32), _p(sol, C.c_uint8))
    if rc:
        raise ValueError(f"oracle_check rc={rc}")
    return sat, sol


def step(inst, X, eta: float, n_steps: int, B=None, *, step_base: int = 0, state=None,
         want_F: bool = True):
    """Run n_steps of fixed-step PGD.  Returns (X_new, F, sat_count, is_solution, first_step).
    ``state`` = (is_solution, first_step) from an earlier call resumes (frozen stay frozen)."""
    B = int(X.shape[1] if B is None else B)
    X = _check_x(inst, X, B).copy()
    F = np.zeros(B, dtype=np.float64) if want_F else None
    sat = np.zeros(B, dtype=np.int32)
    if state is None:
        sol = np.zeros(B, dtype=np.uint8)
        first = np.full(B, -1, dtype=np.int32)
        resume = 0
    else:
        sol = np.ascontiguousarray(state[0], dtype=np.uint8).copy()
        first = np.ascontiguousarray(state[1], dtype=np.int32).copy()
        resume = 1
    args, keep = _inst_args(inst)
    rc = lib().oracle_step(*args, C.c_int32(B), C.c_int64(X.shape[1]), _p(X, C.c_double),
                           C.c_double(eta), C.c_int32(n_steps), C.c_int32(step_base),
                           C.c_int32(resume), _p(F, C.c_double), _p(sat, C.c_int32),
                           _p(sol, C.c_uint8), _p(first, C.c_int32))
    if rc:
        raise ValueError(f"oracle_step rc={rc}")
    return X, F, sat, sol, first


def step_ls(inst, X, n_steps: int, B=None, *, s_max: float = 1.0, beta: float = 0.5, c1: float = 1e-4,
            delta: float = 1e-6, max_trials: int = 8, step_base: int = 0, state=None, want_F: bool = True):
    """Alg. 1 with the backtracking line search of reading B5 (oracle_step_ls).
    Returns (X_new, F, eta, sat_count, is_solution, first_step, converged, margin)."""
    B = int(X.shape[1] if B is None else B)
    X = _check_x(inst, X, B).copy()
    F = np.zeros(B, dtype=np.float64) if want_F else None
    eta = np.zeros(B, dtype=np.float64)
    margin = np.zeros(B, dtype=np.float64)
    sat = np.zeros(B, dtype=np.int32)
    if state is None:
        sol = np.zeros(B, dtype=np.uint8)
        first = np.full(B, -1, dtype=np.int32)
        conv = np.zeros(B, dtype=np.uint8)
        resume = 0
    else:
        sol = np.ascontiguousarray(state[0], dtype=np.uint8).copy()
        first = np.ascontiguousarray(state[1], dtype=np.int32).copy()
        conv = np.ascontiguousarray(state[2], dtype=np.uint8).copy()
        resume = 1
    args, keep = _inst_args(inst)
    rc = lib().oracle_step_ls(*args, C.c_int32(B), C.c_int64(X.shape[1]), _p(X, C.c_double),
                              C.c_double(s_max), C.c_double(beta), C.c_double(c1), C.c_double(delta),
                              C.c_int32(max_trials), C.c_int32(n_steps), C.c_int32(step_base),
                              C.c_int32(resume), _p(F, C.c_double), _p(eta, C.c_double),
                              _p(sat, C.c_int32), _p(sol, C.c_uint8), _p(first, C.c_int32),
                              _p(conv, C.c_uint8), _p(margin, C.c_double))
    if rc:
        raise ValueError(f"oracle_step_ls rc={rc}")
    return X, F, eta, sat, sol, first, conv, margin


def restart(inst, X, seed: int, round_: int, B=None, *, keep=None):
    """Counter-based uniform re-initialisation (oracle_restart); returns a new X."""
    B = int(X.shape[1] if B is None else B)
    X = _check_x(inst, X, B).copy()
    fixed = None if inst.fixed is None else np.ascontiguousarray(inst.fixed, dtype=np.int8)
    keep = None if keep is None else np.ascontiguousarray(keep, dtype=np.uint8)
    rc = lib().oracle_restart(C.c_int32(inst.n_vars), _p(fixed, C.c_int8), C.c_int32(B), C.c_int64(X.shape[1]),
                              _p(X, C.c_double), _p(keep, C.c_uint8), C.c_uint64(seed), C.c_uint32(round_ & 0xFFFFFFFF))
    if rc:
        raise ValueError(f"oracle_restart rc={rc}")
    return X


def solve(inst, X, eta: float, steps_per_round: int, max_rounds: int, seed: int, B=None, *, stop_at_first=True):
    """The restart loop of afsat_solve recomposed from step / restart.  Returns (X, sat, sol, first, rounds)."""
    B = int(X.shape[1] if B is None else B)
    state = None
    r = 0
    sat = None
    while r < max_rounds:
        X, _, sat, sol, first = step(inst, X, eta, steps_per_round, B, step_base=r * steps_per_round, state=state,
                                     want_F=False)
        state = (sol, first)
        any_now = bool(np.any((first > r * steps_per_round)))
        r += 1
        if (any_now and stop_at_first) or r == max_rounds:
            break
        X = restart(inst, X, seed, r - 1, B, keep=sol)
    return X, sat, state[0], state[1], r
