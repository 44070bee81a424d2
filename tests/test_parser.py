"""Problem ingestion (`-m "not gpu"` except the last test): afsat_parse (csrc/parser.cpp, through the C
ABI) and the plain Python reading oracle/parser_oracle.py, both against what PAPER.md App. A fixes:
the paper's own example file with its constraints written out by hand from Table 2,
the CARD normalisation (:264), every automatic simplification of A.1 (:300-309) -- checked by
equisatisfiability with the TEXT's semantics, evaluated here by a third, direct reading -- and each
other; then one GPU test runs a parsed file through afsat_create / afsat_check."""
import itertools
from pathlib import Path

import numpy as np
import pytest

from oracle import parser_oracle as PO
from paper_2606_06641_b200 import binding as Bd
from paper_2606_06641_b200 import build as Build

GOLDEN = Path(__file__).resolve().parent / "golden" / "hybrid_example.txt"
OR, XOR, ATLEAST, ATMOST, EXACTLY, NAE = range(6)


@pytest.fixture(scope="module", autouse=True)
def _built():
    Build.build()


def as_list(pr):
    """Problem (binding) -> the oracle parser's representation."""
    cons = []
    for c in range(pr.n_cons):
        lo, hi = int(pr.row_ptr[c]), int(pr.row_ptr[c + 1])
        cons.append((int(pr.ctype[c]), int(pr.param[c]),
                     tuple((int(v), int(s)) for v, s in zip(pr.lit_var[lo:hi], pr.lit_sign[lo:hi]))))
    fixed = {int(v): int(pr.fixed[v]) for v in np.nonzero(pr.fixed)[0]}
    return {"n_vars": pr.n_vars, "constraints": cons, "fixed": fixed}


def both(text):
    b = PO.parse(text)                                            # raises first when the text is refused
    a = as_list(Bd.parse(text))
    assert a["n_vars"] == b["n_vars"] and a["constraints"] == b["constraints"] and a["fixed"] == b["fixed"]
    return b


# ---- the paper's example, expected values by hand from Table 2 ---------------------------------------
def test_paper_example_file():
    L = lambda *ls: tuple((abs(l) - 1, 1 if l > 0 else -1) for l in ls)   # noqa: E731
    expected = [
        (OR, 0, L(1, -2, 3)), (OR, 0, L(-1, 4)),                  # the DIMACS CNF section
        (OR, 0, L(1, -2, 3)), (XOR, 1, L(1, 2, 3)), (NAE, 0, L(1, 2, 3)), (ATMOST, 1, L(1, 2, 3)),
        (EXACTLY, 1, L(4, 5, 6)), (EXACTLY, 2, L(1, 2, 3)), (ATLEAST, 2, L(1, 2, 3)),
        (ATLEAST, 2, L(1, 2, 3)),                                 # card 2     : >= 2
        (ATMOST, 2, L(1, 2, 3, 4)),                               # card -3    : < 3
        (ATLEAST, 3, L(1, 2, 3, 4)),                              # card >2    : > 2
        (ATMOST, 2, L(1, 2, 3)),                                  # card <=2
    ]
    text = GOLDEN.read_text()
    got = both(text)
    assert got["n_vars"] == 6 and got["fixed"] == {} and got["constraints"] == expected
    pr = Bd.parse_file(GOLDEN)
    assert as_list(pr)["constraints"] == expected
    assert pr.stats["constraints_read"] == 13 and pr.stats["declared_vars"] == 6
    assert pr.stats["declared_constraints"] == 9 and pr.stats["constraints_discarded"] == 0


def test_spellings_and_layout():
    """Short and long identifiers, optional 'h', operator glued to or apart from the threshold, constraints
    spanning lines, '*' comments, a trailing comment after the closing 0."""
    a = both("p cnf 5 4\nh xor 1 2 3 0\nn 1 2 3 0\nh a 1 2 3 0\ne 1 2 3 0\nk 2 1 2 3 0\nd >= 2 1 2 3 0\n")
    b = both("* star comment\np cnf 5 4\nx 1 2\n 3 0 c trailing\nh nae 1 2 3 0\namo 1 2 3 0\nh eo 1 2 3 0\nek 2 1 2 3 0\ncard >=2 1 2 3 0\n")
    assert a == {**b, "read": a["read"], "discarded": a["discarded"]} or a["constraints"] == b["constraints"]
    assert [c[0] for c in a["constraints"]] == [XOR, NAE, ATMOST, EXACTLY, EXACTLY, ATLEAST]
    assert a["n_vars"] == 5                                        # declared variables beyond the used ones stay


# ---- a third, direct reading of the TEXT's semantics (Table 2), used as ground truth ------------------
def text_satisfied(lines, assign):
    """lines: [(ident, thr_string_or_None, [lits])]; assign: dict var(1-based) -> bool.  True iff every
    constraint of the text holds.  Written straight from Table 2 / PAPER.md:264."""
    for ident, thr, lits in lines:
        tau = sum(1 for l in lits if assign[abs(l)] == (l > 0))
        k = len(lits)
        if ident == "":
            ok = tau >= 1
        elif ident in ("x", "xor"):
            ok = tau % 2 == 1
        elif ident in ("n", "nae"):
            ok = 0 < tau < k
        elif ident in ("a", "amo"):
            ok = tau <= 1
        elif ident in ("e", "eo"):
            ok = tau == 1
        elif ident in ("k", "ek"):
            ok = tau == int(thr)
        else:
            if thr.startswith(">="):
                ok = tau >= int(thr[2:])
            elif thr.startswith("<="):
                ok = tau <= int(thr[2:])
            elif thr.startswith(">"):
                ok = tau > int(thr[1:])
            elif thr.startswith("<"):
                ok = tau < int(thr[1:])
            else:
                ok = tau >= int(thr) if int(thr) > 0 else tau < -int(thr)
        if not ok:
            return False
    return True


def parsed_satisfied(parsed, assign):
    for v, val in parsed["fixed"].items():
        if assign[v + 1] != (val == -1):
            return False
    for t, p, lits in parsed["constraints"]:
        tau = sum(1 for v, s in lits if assign[v + 1] == (s > 0))
        k = len(lits)
        ok = {OR: tau >= 1, XOR: tau % 2 == p, ATLEAST: tau >= p, ATMOST: tau <= p, EXACTLY: tau == p,
              NAE: 0 < tau < k}[t]
        if not ok:
            return False
    return True


def render(lines, rng):
    out = ["p cnf 6 %d" % len(lines)]
    for ident, thr, lits in lines:
        w = (["h"] if rng.random() < 0.5 else []) + ([ident] if ident else []) + ([thr] if thr is not None else [])
        out.append(" ".join(w + [str(l) for l in lits] + ["0"]))
    return "\n".join(out) + "\n"


def random_lines(rng, n_vars=6, n_lines=5):
    lines = []
    for _ in range(n_lines):
        k = int(rng.integers(1, 5))
        vs = rng.choice(np.arange(1, n_vars + 1), size=k, replace=False)
        lits = [int(v) * (1 if rng.random() < 0.5 else -1) for v in vs]
        ident = str(rng.choice(["", "x", "xor", "n", "nae", "a", "amo", "e", "eo", "k", "ek", "d", "card"]))
        thr = None
        if ident in ("k", "ek"):
            thr = str(int(rng.integers(0, k + 1)))
        elif ident in ("d", "card"):
            op = str(rng.choice(["", "", ">=", ">", "<=", "<"]))
            if op == "":
                t = int(rng.integers(1, k + 2)) * (1 if rng.random() < 0.6 else -1)
            else:
                t = int(rng.integers(1, k + 2))
            thr = op + str(t)
        lines.append((ident, thr, lits))
    return lines


def test_simplifications_are_equisatisfiable_with_the_text():
    """A.1 (and readings B6): over ALL 2^6 assignments, the text holds iff (prefix assignments hold and
    every kept constraint holds); a text the parsers call UNSAT has no satisfying assignment."""
    rng = np.random.default_rng(66410)
    n_unsat = n_fixed = n_disc = 0
    for trial in range(300):
        lines = random_lines(rng)
        text = render(lines, rng)
        assigns = [dict(zip(range(1, 7), bits)) for bits in itertools.product([False, True], repeat=6)]
        truth = [text_satisfied(lines, a) for a in assigns]
        try:
            parsed = both(text)
        except PO.Unsat:
            with pytest.raises(Bd.AfsatError) as ei:
                Bd.parse(text)
            assert ei.value.code == -9
            # UNSAT on its face is allowed to be reported only if the text really has no model
            assert not any(truth), text
            n_unsat += 1
            continue
        n_fixed += bool(parsed["fixed"]); n_disc += parsed["discarded"] > 0
        assert [parsed_satisfied(parsed, a) for a in assigns] == truth, text
        for t, p, lits in parsed["constraints"]:               # what is kept is what afsat_create accepts
            assert 2 <= len(lits) or t in (XOR, NAE)
            if t in (ATLEAST, ATMOST, EXACTLY):
                assert 0 < p < len(lits)
    assert n_unsat > 5 and n_fixed > 30 and n_disc > 30


def test_each_rule_of_A1():
    P = lambda t: both("p cnf 4 1\n" + t + "\n")               # noqa: E731
    assert P("3 0")["fixed"] == {2: -1} and P("-3 0")["fixed"] == {2: +1}            # unit CNF
    assert P("eo -2 0")["fixed"] == {1: +1}                                          # unit EO
    r = P("amo 2 0"); assert r["fixed"] == {} and r["constraints"] == []             # unit AMO discarded
    assert P("card 1 1 2 3 0")["constraints"] == [(OR, 0, ((0, 1), (1, 1), (2, 1)))] # CARD-1 -> CNF
    assert P("ek 1 1 2 3 0")["constraints"] == [(EXACTLY, 1, ((0, 1), (1, 1), (2, 1)))]   # EK-1 = EO
    assert P("eo 1 2 3 0")["constraints"] == P("ek 1 1 2 3 0")["constraints"]
    assert P("card 3 1 -2 3 0")["fixed"] == {0: -1, 1: +1, 2: -1}                    # CARD-n -> units
    assert P("ek 3 1 -2 3 0")["fixed"] == {0: -1, 1: +1, 2: -1}                      # EK-n -> units
    r = P("card >=1 1 0"); assert r["fixed"] == {0: -1}
    r = P("card <=5 1 2 3 0"); assert r["constraints"] == [] and r["fixed"] == {}    # CARD-0 in '<' form
    assert P("ek 0 1 -2 0")["fixed"] == {0: +1, 1: -1}                               # EK-0 -> negated units
    assert P("card -1 1 2 0")["fixed"] == {0: +1, 1: +1}                             # < 1: none true


def test_errors():
    for text, code in [("p cnf 2 2\n1 0\n-1 0\n", -9),              # contradictory units
                       ("p cnf 3 1\ncard 4 1 2 3 0\n", -9),          # >= 4 of 3
                       ("p cnf 3 1\nek 5 1 2 3 0\n", -9),
                       ("p cnf 3 1\nx 1 1 2 0\n", -5),               # repeated variable outside a disjunction
                       ("p cnf 3 1\nfoo 1 2 0\n", -1),
                       ("p cnf 3 1\n1 2 3\n", -1),                   # not terminated
                       ("p dnf 3 1\n1 2 0\n", -1)]:
        with pytest.raises(Bd.AfsatError) as ei:
            Bd.parse(text)
        assert ei.value.code == code, text
        with pytest.raises(ValueError):
            PO.parse(text)
    r = both("p cnf 3 2\n1 1 -2 0\n2 -2 3 0\n")                   # repeated literal kept once; tautology dropped
    assert r["constraints"] == [(OR, 0, ((0, 1), (1, -1)))]


def test_length_limit_binds_only_emitted_constraints():
    """AFSAT_MAX_LEN (64) applies to what reaches a kernel: a 70-literal constraint that A.1 turns into prefix
    assignments or discards parses; one that stays a constraint is AFSAT_E_LENGTH."""
    lits = " ".join(str(i) for i in range(1, 71))
    for head, fixed_val in (("card >=70", -1), ("ek 70", -1), ("ek 0", +1), ("card <1", +1)):
        pr = Bd.parse(f"p cnf 70 1\n{head} {lits} 0\n")
        assert pr.n_cons == 0 and np.all(pr.fixed == fixed_val), head
    for head in ("card <=70", "card <71", "card <=71"):
        pr = Bd.parse(f"p cnf 70 1\n{head} {lits} 0\n")
        assert pr.n_cons == 0 and not np.any(pr.fixed), head
    for head in ("", "x", "card >=3", "ek 2", "card <5"):
        with pytest.raises(Bd.AfsatError) as ei:
            Bd.parse(f"p cnf 70 1\n{head} {lits} 0\n")
        assert ei.value.code == -2, head


def test_parsed_arrays_are_accepted_by_afsat_create_validation():
    """No device here: afsat_create validates before touching CUDA, so a parsed problem must get past
    validation and fail only with AFSAT_E_CUDA (or succeed on a GPU box)."""
    pr = Bd.parse(GOLDEN.read_text())
    try:
        ctx = pr.context(batch=4)
        ctx.close()
    except Bd.AfsatError as e:
        assert e.code == -8, e


@pytest.mark.gpu
def test_parse_then_check_on_gpu():
    import torch
    from oracle import oracle as O
    from paper_2606_06641_b200 import instances as I
    pr = Bd.parse(GOLDEN.read_text())
    inst = I.Instance(name="paper_example", n_vars=pr.n_vars, row_ptr=pr.row_ptr, lit_var=pr.lit_var, lit_sign=pr.lit_sign,
                      ctype=pr.ctype, param=pr.param, fixed=None, batch=64, eta=0.1, steps=1, meta={})
    B = 64                                                        # all 2^6 assignments as corner candidates
    X = np.zeros((6, 64), dtype=np.float32)
    for b, bits in enumerate(itertools.product([False, True], repeat=6)):
        X[:, b] = [-1.0 if t else 1.0 for t in bits]
    ctx = pr.context(batch=B)
    sat, sol = ctx.check(torch.from_numpy(X).cuda())
    so, solo = O.check(inst, X.astype(np.float64), B)
    assert np.array_equal(sat.cpu().numpy(), so) and np.array_equal(sol.cpu().numpy(), solo)
    F, G = ctx.eval_grad(torch.from_numpy(X).cuda())
    assert np.allclose(F.cpu().numpy(), pr.n_cons - 2.0 * so, atol=1e-4)      # corners: FE = -1 sat / +1 violated
    ctx.close()
