"""Plain Python reading of the paper's input format -- TEST INFRASTRUCTURE ONLY (see oracle.py).

Follows PAPER.md:211-264 (App. A: grammar, Table 2 semantics, CARD normalisation) and PAPER.md:300-309
(A.1 automatic simplification) line by line, with the readings DESIGN.md B6 lists where the paper is
silent.  It shares nothing with the product parser (csrc/parser.cpp) and never imports the product
package.  Pins (tests/test_parser.py): the paper's own example file (tests/golden/hybrid_example.txt,
expected constraints written out by hand from Table 2) and, for every A.1 rule, equisatisfiability of
the simplified output with the text's own semantics over all assignments of small instances.

parse(text) -> dict(n_vars, constraints=[(type, param, ((var0, sign), ...)), ...], fixed={var0: -1|+1},
                    read, discarded)
types: 0 OR, 1 XOR (param = parity), 2 ATLEAST, 3 ATMOST, 4 EXACTLY, 5 NAE; var0 is 0-based;
sign +1: literal true iff the variable is True; fixed: -1 = True, +1 = False (True <-> -1).
"""
from __future__ import annotations

OR, XOR, ATLEAST, ATMOST, EXACTLY, NAE = range(6)
MAX_LEN = 64


class Unsat(ValueError):
    pass


class Duplicate(ValueError):
    pass


def _is_int(tok: str) -> bool:
    body = tok[1:] if tok[:1] in "+-" else tok
    return body.isdigit()


def parse(text: str) -> dict:
    words = []                                        # comment LINES vanish, the rest is one token stream
    for line in text.splitlines():
        w = line.split()
        if not w or w[0] == "c" or w[0].startswith("*"):
            continue
        # a comment may follow the closing 0 on the same line
        for i, tok in enumerate(w):
            if i > 0 and w[i - 1] == "0" and (tok == "c" or tok.startswith("*")):
                w = w[:i]
                break
        words.extend(w)
    n_vars, declared = 0, 0
    cons, fixed = [], {}
    read = discarded = 0

    def assign(var, sign, lit_true):
        val = -1 if ((sign > 0) == lit_true) else +1
        if fixed.get(var, val) != val:
            raise Unsat("contradictory unit assignments")
        fixed[var] = val

    i = 0
    while i < len(words):
        if words[i] == "p":
            if words[i + 1] != "cnf":
                raise ValueError("p line")
            declared = max(declared, int(words[i + 2]))
            int(words[i + 3])
            i += 4
            continue
        if words[i] == "h":
            i += 1
        kind, thr = "cnf", None
        if not _is_int(words[i]):
            ident = words[i]
            i += 1
            kind = {"x": "xor", "xor": "xor", "n": "nae", "nae": "nae", "a": "amo", "amo": "amo",
                    "e": "eo", "eo": "eo", "k": "ek", "ek": "ek", "d": "card", "card": "card"}.get(ident)
            if kind is None:
                raise ValueError(f"unknown identifier {ident!r}")
            if kind == "ek":
                thr = int(words[i]); i += 1
            elif kind == "card":
                tok = words[i]; i += 1
                op = ""
                for cand in ("<=", ">=", "<", ">"):
                    if tok.startswith(cand):
                        op, tok = cand, tok[len(cand):]
                        break
                if op and tok == "":
                    tok = words[i]; i += 1
                kk = int(tok)
                if op and kk < 1:
                    raise ValueError("card threshold")
                if not op and kk == 0:
                    raise ValueError("card threshold")
                # normalise to (>= a) or (<= b) on the count of true literals
                if op == "":
                    thr = (">=", kk) if kk > 0 else ("<=", -kk - 1)
                elif op == ">=":
                    thr = (">=", kk)
                elif op == ">":
                    thr = (">=", kk + 1)
                elif op == "<=":
                    thr = ("<=", kk)
                else:
                    thr = ("<=", kk - 1)
        lits = []
        while True:
            if i >= len(words):
                raise ValueError("constraint not terminated by 0")
            l = int(words[i]); i += 1
            if l == 0:
                break
            lits.append((abs(l) - 1, 1 if l > 0 else -1))
            n_vars = max(n_vars, abs(l))
        read += 1
        if not lits:
            raise ValueError("empty constraint")
        if kind == "cnf":
            uniq = []
            taut = False
            for v, s in lits:
                if (v, -s) in uniq:
                    taut = True
                if (v, s) not in uniq:
                    uniq.append((v, s))
            if taut:
                discarded += 1
                continue
            lits = uniq
        elif len({v for v, _ in lits}) != len(lits):
            raise Duplicate("repeated variable")
        k = len(lits)
        if k > MAX_LEN:
            raise ValueError("too long")
        # Table 2 -> (lo, hi) window on the number of true literals where that exists
        if kind == "cnf":
            win = (1, k)
        elif kind == "amo":
            win = (0, 1)
        elif kind == "eo":
            win = (1, 1)
        elif kind == "ek":
            win = (thr, thr)
        elif kind == "card":
            win = (thr[1], k) if thr[0] == ">=" else (0, thr[1])
        else:
            win = None
        if win is None:
            cons.append((XOR, 1, tuple(lits)) if kind == "xor" else (NAE, 0, tuple(lits)))
            continue
        lo, hi = win
        exact = kind in ("eo", "ek")
        lower = kind in ("cnf",) or (kind == "card" and thr[0] == ">=")
        if exact:
            if lo < 0 or lo > k:
                raise Unsat("exactly-k out of range")
            if lo == k:                               # EK-n, unit EO -> all true
                for v, s in lits:
                    assign(v, s, True)
            elif lo == 0:                             # EK-0 -> all false
                for v, s in lits:
                    assign(v, s, False)
            else:
                cons.append((EXACTLY, lo, tuple(lits)))
        elif lower:
            if lo <= 0:                               # CARD-0
                discarded += 1
            elif lo > k:
                raise Unsat("at-least above length")
            elif lo == k:                             # CARD-n, unit CNF
                for v, s in lits:
                    assign(v, s, True)
            elif lo == 1:                             # CARD-1 -> CNF
                cons.append((OR, 0, tuple(lits)))
            else:
                cons.append((ATLEAST, lo, tuple(lits)))
        else:                                         # at most hi
            if hi < 0:
                raise Unsat("at-most below zero")
            if hi >= k:                               # unit AMO and friends
                discarded += 1
            elif hi == 0:
                for v, s in lits:
                    assign(v, s, False)
            else:
                cons.append((ATMOST, hi, tuple(lits)))
    n_vars = max(n_vars, declared)
    if n_vars < 1:
        raise ValueError("no variables")
    return {"n_vars": n_vars, "constraints": cons, "fixed": fixed, "read": read, "discarded": discarded}
