"""CPU-side tests of the CUDA library (`-m "not gpu"`): the C ABI loads and exports every symbol
include/afsat.h declares, the host precompute (tailored DFT tables) is pinned
against mathematics that does not involve the library (corner linear system P10, the expectation
identity), input validation reports the documented error codes before any device is touched,
and there is no CPU fallback.  No compute kernel is called here."""
import ctypes
import re
from pathlib import Path

import numpy as np
import pytest

from paper_2606_06641_b200 import binding as Bd
from paper_2606_06641_b200 import build as Build
from paper_2606_06641_b200 import instances as I
from tests import refmath as R

ROOT = Path(__file__).resolve().parents[1]
ALL_TYPES = [R.OR, R.XOR, R.ATLEAST, R.ATMOST, R.EXACTLY, R.NAE]
rng0 = np.random.default_rng(424242)


@pytest.fixture(scope="module", autouse=True)
def _built():
    Build.build()


def test_header_symbols_exported():
    text = (ROOT / "include" / "afsat.h").read_text()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    declared = sorted(set(re.findall(r"\b(afsat_[a-z_]+)\s*\(", text)))
    assert set(declared) == set(Bd.EXPORTS), declared
    lib = ctypes.CDLL(str(Bd.LIB_PATH))
    for name in declared:
        assert hasattr(lib, name), name
    assert "sm_100a" in Bd.version()


def _eval_tables(rows, y):
    """FE and gradient from a table, straight from the contract in afsat.h (numpy complex)."""
    y = np.asarray(y, dtype=np.longdouble)
    fe = np.longdouble(0)
    g = np.zeros(y.shape[0], dtype=np.longdouble)
    for r in rows:
        a = complex(r[0], r[1]); b = complex(r[2], r[3]); w = complex(r[4], r[5]); wb = complex(r[6], r[7])
        f = np.array([a + b * complex(float(v)) for v in y])
        fe += (w * np.prod(f)).real
        for i in range(len(y)):
            g[i] += (wb * np.prod(np.delete(f, i))).real
    return fe, g


def _cases(kmax):
    for k in range(1, kmax + 1):
        for t in ALL_TYPES:
            for p in R.all_params(t, k):
                yield t, k, p


@pytest.mark.parametrize("flags", [Bd.FLAG_DEFAULT, Bd.FLAG_ROBUST])
def test_P10_tables_reproduce_truth_table_at_corners(flags):
    """sum_p Re(w_p prod_i(a_p + b_p y_i)) = g(tau) at a corner with tau true literals."""
    for t, k, p in _cases(24):
        if k > 9 and p not in (0, 1, k // 2, k):
            continue
        rows, n_real = Bd.host_tables(t, k, p, flags)
        assert rows.shape[0] <= (k + 1) // 2 + 1
        for tau in range(k + 1):
            y = np.ones(k)
            y[:tau] = -1.0
            fe, _ = _eval_tables(rows, y)
            want = -1.0 if R.is_sat(t, k, p, tau) else 1.0
            assert abs(float(fe) - want) < 1e-9 * 2 ** (k / 2), (t, k, p, tau, float(fe))


@pytest.mark.parametrize("flags", [Bd.FLAG_DEFAULT, Bd.FLAG_ROBUST])
def test_tables_match_expectation_identity_and_gradient(flags):
    for t, k, p in _cases(40):
        if k > 8 and (k % 5 or p not in (0, 1, k // 3, k // 2, k)):
            continue
        rows, n_real = Bd.host_tables(t, k, p, flags)
        y = rng0.uniform(-1, 1, size=k)
        fe, g = _eval_tables(rows, y)
        want = R.fe_expectation(t, k, p, y)
        assert abs(float(fe - want)) < 1e-11, (t, k, p)
        for i in rng0.permutation(k)[:3]:
            yp, ym = y.copy(), y.copy()
            yp[i], ym[i] = 1.0, -1.0
            d = (R.fe_expectation(t, k, p, yp) - R.fe_expectation(t, k, p, ym)) / 2
            assert abs(float(g[i] - d)) < 1e-11, (t, k, p, i)


def test_table_structure_tailored_dft():
    """Paper mode: a = 1/2, b = w^l / 2 with |b| = 1/2 and the roots exactly symmetric: real rows
    have zero imaginary parts, w^(N/4) = i exactly, mirrored rows share |Re b|, |Im b| bit for bit
    (PAPER.md:143-147)."""
    for k in (3, 7, 11, 15, 31, 50, 63):
        rows, n_real = Bd.host_tables(R.EXACTLY, k, k // 2, 0)
        assert np.all(rows[:, 0] == 0.5) and np.all(rows[:, 1] == 0.0)
        assert np.all(rows[:n_real, [1, 3, 5, 7]] == 0.0)
        assert np.allclose(np.hypot(rows[:, 2], rows[:, 3]), 0.5, rtol=0, atol=1e-16)
        bs = {(abs(r[2]), abs(r[3])) for r in rows[n_real:]}
        for br, bi in list(bs):
            if (k + 1) % 4 == 0:         # the point l and its mirror N/2 - l are both present
                assert (br, bi) in bs and ((bi, br) in bs or br == bi or br == 0 or bi == 0)
        if (k + 1) % 4 == 0:
            assert any(r[2] == 0.0 and r[3] == 0.5 for r in rows), "w^(N/4) must be exactly i"


def test_zero_weight_points_are_dropped():
    rows, n_real = Bd.host_tables(R.OR, 3, 0, 0)          # d = (0, -1/4, -1/4, -1/4): l = 0 vanishes
    assert rows.shape[0] == 2 and n_real == 1
    rows, n_real = Bd.host_tables(R.ATLEAST, 3, 2, 0)     # d = (0, -i/4, 0, i/4)
    assert rows.shape[0] == 1 and n_real == 0
    assert np.array_equal(rows[0], [0.5, 0, 0, 0.5, 0, -4, 2, 0])


def test_host_tables_rejects():
    tab = np.zeros(33 * 8)
    L = Bd.load_library()
    assert L.afsat_host_tables(0, 0, 0, 0, tab.ctypes.data, None) == -2
    assert L.afsat_host_tables(0, 65, 0, 0, tab.ctypes.data, None) == -2
    assert L.afsat_host_tables(9, 3, 0, 0, tab.ctypes.data, None) == -1
    assert L.afsat_host_tables(2, 3, 4, 0, tab.ctypes.data, None) == -6
    assert L.afsat_host_tables(1, 3, 2, 0, tab.ctypes.data, None) == -6
    assert L.afsat_host_tables(0, 3, 0, 0, None, None) == -1


def test_restriction_under_a_partial_assignment():
    """afsat_host_restrict (the substitution afsat_create applies) against the test's own predicate: for every
    type, length <= 9, parameter and split of the fixed literals into true / false, the restricted truth table is the
    original one shifted by the fixed-true count, and "decided" means constant."""
    for t, k, p in _cases(9):
        for f_true in range(k + 1):
            for f_false in range(k + 1 - f_true):
                status, kf, mask = Bd.host_restrict(t, k, p, f_true, f_false)
                assert kf == k - f_true - f_false
                want = [R.is_sat(t, k, p, tau + f_true) for tau in range(kf + 1)]
                assert [bool(mask >> tau & 1) for tau in range(kf + 1)] == want and mask >> (kf + 1) == 0
                assert status == (1 if all(want) else 2 if not any(want) else 0)
    with pytest.raises(Bd.AfsatError):
        Bd.host_restrict(R.OR, 3, 0, 2, 2)


@pytest.mark.parametrize("flags", [Bd.FLAG_DEFAULT, Bd.FLAG_ROBUST])
def test_tables_of_restricted_signatures_reproduce_their_truth_table(flags):
    """P10 for the signatures substitution creates (arbitrary symmetric truth tables, e.g. "2 <= tau <= 4 of 6" from an
    EXACTLY / ATLEAST mix): sum_p Re(w_p prod_i (a_p + b_p y_i)) = -1 / +1 at the corner with tau true literals."""
    rng = np.random.default_rng(77)
    for k in (1, 2, 3, 5, 8, 12, 17):
        for _ in range(6):
            mask = int(rng.integers(1, (1 << (k + 1)) - 1))            # non-constant truth table
            rows, n_real = Bd.host_tables_mask(k, mask, flags)
            for tau in range(k + 1):
                y = np.array([-1.0] * tau + [1.0] * (k - tau))
                fe, _ = _eval_tables(rows, y)
                assert abs(float(fe) - (-1.0 if mask >> tau & 1 else 1.0)) < 1e-9, (k, mask, tau, float(fe))
    # the restriction of a Table 1 constraint gets the SAME table as the native constraint with that truth table
    status, kf, mask = Bd.host_restrict(R.OR, 8, 0, 0, 2)
    assert status == 0 and kf == 6
    assert np.array_equal(Bd.host_tables_mask(kf, mask)[0], Bd.host_tables(R.OR, 6, 0)[0])
    status, kf, mask = Bd.host_restrict(R.ATLEAST, 12, 6, 2, 1)        # "at least 6 of 12" -> "at least 4 of 9"
    assert np.array_equal(Bd.host_tables_mask(kf, mask)[0], Bd.host_tables(R.ATLEAST, 9, 4)[0])


def _has_gpu():
    import torch
    return torch.cuda.is_available()


def _create(inst, **kw):
    return Bd.Context.from_instance(inst, **kw)


def test_create_validation_codes():
    base = I.make_mixed(n=12, m=6, kmin=2, kmax=5, seed=3, batch=4)

    def mutated(**changes):
        d = dict(base.__dict__)
        for k_, v in changes.items():
            d[k_] = v
        return I.Instance(**d)

    def expect(code, inst, **kw):
        with pytest.raises(Bd.AfsatError) as ei:
            _create(inst, **kw)
        assert ei.value.code == code, (ei.value.code, str(ei.value))

    lv = base.lit_var.copy(); lv[1] = lv[0]
    expect(-5, mutated(lit_var=lv))                                   # duplicate variable (A15)
    lv = base.lit_var.copy(); lv[0] = 12
    expect(-3, mutated(lit_var=lv))
    lv = base.lit_var.copy(); lv[0] = -1
    expect(-3, mutated(lit_var=lv))
    ls = base.lit_sign.copy(); ls[2] = 0
    expect(-4, mutated(lit_sign=ls))
    ty = base.ctype.copy(); ty[0] = 6
    expect(-1, mutated(ctype=ty))
    ty = base.ctype.copy(); ty[0] = R.ATLEAST
    pa = base.param.copy(); pa[0] = 99
    expect(-6, mutated(ctype=ty, param=pa))
    pa = base.param.copy(); pa[0] = -1
    expect(-6, mutated(ctype=ty, param=pa))
    fx = np.zeros(12, dtype=np.int8); fx[3] = 2
    expect(-4, mutated(fixed=fx))
    expect(-1, base, batch=0)
    expect(-1, base, batch=4, ldb=48)                                  # ldb % 32 != 0
    expect(-1, base, batch=40, ldb=32)                                 # ldb < B
    expect(-1, base, dtype=16)
    expect(-1, base, flags=8)
    expect(-1, base, flags=Bd.FLAG_ROBUST | Bd.FLAG_PAPER)             # the two table modes exclude each other
    # afsat_create_ex options (include/afsat.h): explicit tile width, step path, several partial assignments
    expect(-1, base, tile_w=48)                                        # not a multiple of 32
    expect(-1, base, step_path=7)
    masks = np.zeros((2, 12), dtype=np.int8); masks[0, 1] = 1
    expect(-1, base, batch=96, fixed=masks)                            # 96 % (32 * 2) != 0
    expect(-8, base, batch=128, fixed=masks) if not _has_gpu() else None   # valid: fails only for want of a device
    bad = masks.copy(); bad[1, 5] = 3
    expect(-4, base, batch=128, fixed=bad)
    # constraint longer than AFSAT_MAX_LEN / empty constraint
    n = 80
    rp = np.array([0, 65], dtype=np.int64)
    long_ = I.Instance("long", n, rp, np.arange(65, dtype=np.int32), np.ones(65, dtype=np.int8),
                       np.array([0], dtype=np.uint8), np.array([0], dtype=np.int32), batch=4)
    expect(-2, long_)
    rp = np.array([0, 0], dtype=np.int64)
    empty = I.Instance("empty", n, rp, np.zeros(0, dtype=np.int32), np.zeros(0, dtype=np.int8),
                       np.array([0], dtype=np.uint8), np.array([0], dtype=np.int32), batch=4)
    expect(-2, empty)


def test_no_cpu_fallback():
    """Without a CUDA device the product path fails loudly with AFSAT_E_CUDA."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    inst = I.make_config(0)
    with pytest.raises(Bd.AfsatError) as ei:
        _create(inst)
    assert ei.value.code == -8 and "no CPU fallback" in str(ei.value)


def test_product_does_not_import_oracle():
    """The package (and the C sources) never reference oracle/; the oracle never references them."""
    pat = re.compile(r"(import\s+oracle|from\s+oracle|oracle[./\\]|liboracle|oracle_[a-z_]+\s*\()")
    for p in list((ROOT / "paper_2606_06641_b200").rglob("*")) + list((ROOT / "include").glob("*")):
        if p.suffix in (".py", ".cu", ".cuh", ".cpp", ".h"):
            assert not pat.search(p.read_text()), p
    for p in (ROOT / "oracle").glob("*"):
        if p.suffix in (".py", ".c"):
            txt = p.read_text()
            assert "import paper_2606" not in txt and "from paper_2606" not in txt and "afsat.h" not in txt, p


def test_generators_are_deterministic_and_shaped():
    a, b = I.make_config(2, scale=0.05), I.make_config(2, scale=0.05)
    for f in ("row_ptr", "lit_var", "lit_sign", "ctype", "param", "fixed"):
        assert np.array_equal(getattr(a, f), getattr(b, f))
    c0 = I.make_config(0)
    assert (c0.n_vars, c0.n_cons, c0.nnz, c0.batch) == (50, 213, 639, 64)
    c1 = I.make_config(1, scale=0.01)
    assert set(c1.lengths()) == {7} and set(np.unique(c1.ctype)) == {R.OR}
    c3 = I.make_config(3, scale=0.05)
    ks = c3.lengths()
    assert ks.min() >= 30 and ks.max() <= 50
    assert np.all(c3.param >= -(-ks // 4)) and np.all(c3.param <= 3 * ks // 4)
    c4 = I.make_config(4, scale=0.01)
    assert set(np.unique(c4.ctype)) == {R.OR, R.XOR, R.NAE} and c4.lengths().max() <= 5
    for inst in (a, c0, c1, c3, c4):                       # variables distinct inside a constraint
        for c in rng0.integers(0, inst.n_cons, size=50):
            v = inst.lit_var[inst.row_ptr[c]:inst.row_ptr[c + 1]]
            assert len(set(v.tolist())) == len(v)
        assert set(np.unique(inst.lit_sign)) <= {-1, 1}
    x = I.make_x0(a, batch=40)
    assert x.shape == (a.n_vars, 64) and x.dtype == np.float32 and np.all(x[:, 40:] == 0)
    fx = a.fixed != 0
    assert abs(fx.mean() - 0.2) < 1e-9 and np.all(x[fx, :40] == a.fixed[fx][:, None])
    assert np.all(np.abs(x) <= 1)
