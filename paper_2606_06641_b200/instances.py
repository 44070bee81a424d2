"""Seeded synthetic input generators shared by the CPU oracle's tests and the CUDA path.

This module holds NONE of the method's arithmetic (no Fourier coefficients, no FE, no
gradient, no satisfaction predicate): it only draws constraint tables, masks and starting
points.  It imports numpy only, so the tests of the CPU oracle and the users of the CUDA binding can
consume exactly the same arrays.

The paper's own workloads (hard random k-SAT; the random-cardinality and
parity-learning sets of its ref. [3]) are not available; the five
configurations of BASELINE.json ``configs`` stand in for them.

Constraint-type enum (mirrors include/afsat.h, semantics from PAPER.md Table 1 :87-97 and
Table 2 :252-262): OR=0, XOR=1, ATLEAST=2, ATMOST=3, EXACTLY=4, NAE=5.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field
from typing import Optional

import numpy as np

OR, XOR, ATLEAST, ATMOST, EXACTLY, NAE = 0, 1, 2, 3, 4, 5
TYPE_NAMES = {OR: "OR", XOR: "XOR", ATLEAST: "ATLEAST", ATMOST: "ATMOST",
              EXACTLY: "EXACTLY", NAE: "NAE"}

SEED_INSTANCE = 6641000
SEED_X0 = 6641100
SEED_MASK = 6641200


@dataclass
class Instance:
    """A CSR constraint table plus an optional partial assignment and a default batch."""
    name: str
    n_vars: int
    row_ptr: np.ndarray        # int64 [m+1]
    lit_var: np.ndarray        # int32 [nnz], 0-based variable index
    lit_sign: np.ndarray       # int8  [nnz], +1 or -1 (literal value y = sign * x)
    ctype: np.ndarray          # uint8 [m]
    param: np.ndarray          # int32 [m]
    fixed: Optional[np.ndarray] = None   # int8 [n]: 0 free, -1 fixed True (x=-1), +1 fixed False
    batch: int = 64
    eta: float = 0.1
    steps: int = 1
    meta: dict = field(default_factory=dict)

    @property
    def n_cons(self) -> int:
        return int(self.row_ptr.shape[0] - 1)

    @property
    def nnz(self) -> int:
        return int(self.lit_var.shape[0])

    def lengths(self) -> np.ndarray:
        return np.diff(self.row_ptr).astype(np.int64)


def _draw_subsets(rng: np.random.Generator, n: int, k: int, count: int) -> np.ndarray:
    """`count` uniform k-subsets of range(n) without replacement, in random order.

    Draw k independent uniform indices per row and redraw the rows that contain a repeat
    (SURVEY.md §8(d)); conditional on no repeat the row is a uniform ordered k-subset.
    """
    if k > n:
        raise ValueError(f"cannot draw {k} distinct variables out of {n}")
    if k * k > 2 * n:
        # rejection would rarely succeed: take the first k entries of a uniform permutation per row
        return np.argsort(rng.random((count, n)), axis=1)[:, :k].astype(np.int32)
    out = rng.integers(0, n, size=(count, k), dtype=np.int64)
    if k == 1:
        return out.astype(np.int32)
    while True:
        srt = np.sort(out, axis=1)
        bad = np.nonzero((srt[:, 1:] == srt[:, :-1]).any(axis=1))[0]
        if bad.size == 0:
            break
        out[bad] = rng.integers(0, n, size=(bad.size, k), dtype=np.int64)
    return out.astype(np.int32)


def _assemble(name, n, groups, rng, *, batch, eta, steps, fixed=None, shuffle=True, meta=None):
    """groups: list of (ctype, lengths[int array], params[int array]). Draw variables and signs."""
    ks = np.concatenate([np.asarray(g[1], dtype=np.int64) for g in groups])
    ty = np.concatenate([np.full(len(g[1]), g[0], dtype=np.uint8) for g in groups])
    pa = np.concatenate([np.asarray(g[2], dtype=np.int32) for g in groups])
    m = ks.shape[0]
    if shuffle and len(groups) > 1:
        perm = rng.permutation(m)
        ks, ty, pa = ks[perm], ty[perm], pa[perm]
    row_ptr = np.zeros(m + 1, dtype=np.int64)
    np.cumsum(ks, out=row_ptr[1:])
    nnz = int(row_ptr[-1])
    lit_var = np.empty(nnz, dtype=np.int32)
    for k in np.unique(ks):
        rows = np.nonzero(ks == k)[0]
        sub = _draw_subsets(rng, n, int(k), rows.size)
        idx = row_ptr[rows][:, None] + np.arange(int(k))[None, :]
        lit_var[idx] = sub
    lit_sign = (rng.integers(0, 2, size=nnz, dtype=np.int8) * 2 - 1).astype(np.int8)
    return Instance(name=name, n_vars=n, row_ptr=row_ptr, lit_var=lit_var, lit_sign=lit_sign,
                    ctype=ty, param=pa, fixed=fixed, batch=batch, eta=eta, steps=steps,
                    meta=dict(meta or {}))


def _scaled(x: int, scale: float, lo: int = 1) -> int:
    return max(lo, int(round(x * scale)))


def make_config(cfg: int, *, scale: float = 1.0, batch: Optional[int] = None,
                instance_seed: Optional[int] = None) -> Instance:
    """BASELINE.json ``configs[cfg]`` as arrays.

    ``scale`` < 1 shrinks the constraint counts (not the lengths, types or ratios) so that the
    CPU oracle finishes quickly; ``batch`` overrides B.  Seeds follow SURVEY.md §8(d).
    """
    seed = SEED_INSTANCE + cfg if instance_seed is None else instance_seed
    rng = np.random.default_rng(seed)
    if cfg == 0:
        n, m = 50, 213
        inst = _assemble("cfg0_3sat_n50", n, [(OR, np.full(m, 3), np.zeros(m))], rng,
                         batch=64, eta=0.1, steps=200)
    elif cfg == 1:
        n = _scaled(2000, scale, 16)
        m = _scaled(170000, scale)
        inst = _assemble("cfg1_7sat_n2000", n, [(OR, np.full(m, 7), np.zeros(m))], rng,
                         batch=1024, eta=0.1, steps=1000)
    elif cfg == 2:
        n = _scaled(5000, scale, 64)
        m_or, m_x, m_al, m_ex = (_scaled(15000, scale), _scaled(3000, scale),
                                 _scaled(1000, scale), _scaled(500, scale))
        k_or = rng.integers(3, 9, size=m_or)
        k_x = rng.integers(3, 7, size=m_x)
        p_x = rng.integers(0, 2, size=m_x)
        k_al = rng.integers(10, 21, size=m_al)
        t_al = (k_al + 1) // 2
        k_ex = np.full(m_ex, 12)
        t_ex = rng.integers(3, 10, size=m_ex)
        mrng = np.random.default_rng(SEED_MASK + cfg)
        fixed = np.zeros(n, dtype=np.int8)
        nfix = n // 5
        which = mrng.choice(n, size=nfix, replace=False)
        fixed[which] = (mrng.integers(0, 2, size=nfix) * 2 - 1).astype(np.int8)
        inst = _assemble("cfg2_hetero_n5000", n,
                         [(OR, k_or, np.zeros(m_or)), (XOR, k_x, p_x),
                          (ATLEAST, k_al, t_al), (EXACTLY, k_ex, t_ex)], rng,
                         batch=4096, eta=0.1, steps=200, fixed=fixed)
    elif cfg == 3:
        n = _scaled(1000, scale, 64)
        half = _scaled(1000, scale)
        ks = rng.integers(30, 51, size=2 * half)
        lo = -(-ks // 4)              # ceil(k/4)
        hi = (3 * ks) // 4            # floor(3k/4)
        ts = lo + (rng.random(2 * half) * (hi - lo + 1)).astype(np.int64)
        inst = _assemble("cfg3_long_card_n1000", n,
                         [(ATLEAST, ks[:half], ts[:half]), (ATMOST, ks[half:], ts[half:])], rng,
                         batch=2048, eta=0.1, steps=100)
    elif cfg == 4:
        n = _scaled(100000, scale, 64)
        m_or, m_x, m_n = _scaled(357000, scale), _scaled(42000, scale), _scaled(21000, scale)
        inst = _assemble("cfg4_large_hetero_n100000", n,
                         [(OR, rng.integers(3, 6, size=m_or), np.zeros(m_or)),
                          (XOR, rng.integers(3, 5, size=m_x), np.ones(m_x)),
                          (NAE, np.full(m_n, 4), np.zeros(m_n))], rng,
                         batch=8192, eta=0.1, steps=500)
    else:
        raise ValueError(f"unknown config {cfg}")
    if batch is not None:
        inst.batch = int(batch)
    inst.meta.update(cfg=cfg, scale=scale, seed=seed)
    return inst


def make_mixed(n: int, m: int, *, kmin: int = 1, kmax: int = 12, seed: int = 1,
               batch: int = 64, with_fixed: bool = False, types=None) -> Instance:
    """A small instance with every constraint type, lengths uniform in [kmin,kmax] and parameters
    covering the whole admissible range (including the trivial t=0 and t=k) - used by edge-case
    and parity tests, not by the benchmark."""
    rng = np.random.default_rng(seed)
    types = list(types) if types is not None else [OR, XOR, ATLEAST, ATMOST, EXACTLY, NAE]
    ty = rng.choice(np.asarray(types, dtype=np.uint8), size=m)
    ks = rng.integers(kmin, min(kmax, n) + 1, size=m)
    pa = np.zeros(m, dtype=np.int32)
    for j in range(m):
        if ty[j] == XOR:
            pa[j] = rng.integers(0, 2)
        elif ty[j] in (ATLEAST, ATMOST, EXACTLY):
            pa[j] = rng.integers(0, ks[j] + 1)
    fixed = None
    if with_fixed:
        fixed = np.zeros(n, dtype=np.int8)
        which = rng.choice(n, size=max(1, n // 5), replace=False)
        fixed[which] = (rng.integers(0, 2, size=which.size) * 2 - 1).astype(np.int8)
    groups = [(int(ty[j]), np.array([ks[j]]), np.array([pa[j]])) for j in range(m)]
    return _assemble(f"mixed_n{n}_m{m}", n, groups, rng, batch=batch, eta=0.1, steps=20,
                     fixed=fixed, shuffle=False)


def make_x0(inst: Instance, *, seed: Optional[int] = None, batch: Optional[int] = None,
            ldb: Optional[int] = None, dtype=np.float32) -> np.ndarray:
    """Starting points, variable-major ``x[v, b]`` (shape [n, ldb]), uniform in [-1,1) drawn in
    fp32 (``2*rng.random(float32)-1``) and widened exactly when ``dtype`` is float64.  Rows of
    fixed variables hold the fixed value for every candidate.  Padding columns
    (b >= B) are zero."""
    B = int(batch if batch is not None else inst.batch)
    ldb = int(ldb if ldb is not None else padded_ldb(B))
    cfg = inst.meta.get("cfg", 0)
    rng = np.random.default_rng(SEED_X0 + cfg if seed is None else seed)
    x = np.zeros((inst.n_vars, ldb), dtype=np.float32)
    x[:, :B] = 2.0 * rng.random((inst.n_vars, B), dtype=np.float32) - 1.0
    if inst.fixed is not None:
        fx = inst.fixed != 0
        x[fx, :B] = inst.fixed[fx].astype(np.float32)[:, None]
    return x.astype(dtype)


def padded_ldb(B: int) -> int:
    """Leading dimension: B rounded up to a multiple of 32 (128-byte rows in fp32)."""
    return (int(B) + 31) // 32 * 32


def corner_x(inst: Instance, assignment_true: np.ndarray, *, ldb: Optional[int] = None,
             dtype=np.float32) -> np.ndarray:
    """x[v,b] = -1 where assignment_true[v,b] else +1 (True -> -1)."""
    n, B = assignment_true.shape
    ldb = int(ldb if ldb is not None else padded_ldb(B))
    x = np.zeros((n, ldb), dtype=dtype)
    x[:, :B] = np.where(assignment_true, -1.0, 1.0)
    return x


def plant_solution(inst: Instance, *, seed: int = 7):
    """Return (instance', hidden) where the literal signs of `inst` are re-chosen so that the
    hidden Boolean assignment satisfies every constraint.

    For each constraint a target number tau of true literals is chosen among the counts that
    the caller-supplied admissible set allows; the admissible sets are passed in by the caller
    through ``inst.meta['admissible']`` (a list of arrays of allowed tau per constraint) so that
    this module stays free of the satisfaction predicate.
    """
    rng = np.random.default_rng(seed)
    adm = inst.meta["admissible"]
    hidden = rng.integers(0, 2, size=inst.n_vars).astype(bool)   # True = variable is True
    if inst.fixed is not None:
        fx = inst.fixed != 0
        hidden[fx] = inst.fixed[fx] < 0
    sign = inst.lit_sign.copy()
    for c in range(inst.n_cons):
        lo, hi = int(inst.row_ptr[c]), int(inst.row_ptr[c + 1])
        k = hi - lo
        tau = int(rng.choice(np.asarray(adm[c])))
        want_true = np.zeros(k, dtype=bool)
        want_true[rng.permutation(k)[:tau]] = True
        var_true = hidden[inst.lit_var[lo:hi]]
        # literal true iff (sign=+1 and var True) or (sign=-1 and var False)
        sign[lo:hi] = np.where(want_true == var_true, 1, -1).astype(np.int8)
    out = Instance(name=inst.name + "_planted", n_vars=inst.n_vars, row_ptr=inst.row_ptr,
                   lit_var=inst.lit_var, lit_sign=sign, ctype=inst.ctype, param=inst.param,
                   fixed=inst.fixed, batch=inst.batch, eta=inst.eta, steps=inst.steps,
                   meta=dict(inst.meta))
    return out, hidden
