// parser.cpp -- problem ingestion (SURVEY.md §1 layer L1, §8(f) NEXT #2): DIMACS CNF and the paper's
// DIMACS-like hybrid PB format (App. A) with the automatic simplifications of
// PAPER.md:300-309 (A.1), producing exactly what afsat_create consumes: a CSR constraint table
// (row_ptr, lit_var, lit_sign, type, param) and the partial-assignment mask fixed[].
//
// Grammar (tokens are whitespace-separated, a constraint ends with the token 0 and
// may span lines):  comment 'c' / '*' <text> ;  problem 'p cnf <V> <C>' ;
//   constraint  ['h'] ( <lit>+ | (x|xor|n|nae|a|amo|e|eo) <lit>+ | (k|ek) <int> <lit>+
//                      | (d|card) [<|<=|>|>=]<int> <lit>+ )  0
// Semantics (Table 2; CARD normalisation :264): plain = disjunction, xor = odd
// number of true literals, nae = not all equal, amo = at most one, eo = exactly one, ek = exactly k,
// card with a bare threshold: k > 0 means >= k, k < 0 means < |k|; '>' k is >= k+1, '<' k is <= k-1.
// Literal l: variable |l| (1-based), true iff the variable is True (l > 0) or False (l < 0).
//
// Simplifications (A.1, applied once per constraint as it is read -- the paper describes no fixpoint):
//   unit EO / CNF -> prefix assignment;  unit AMO -> discarded;  CARD-1 -> CNF;  EK-1 -> EO;
//   CARD-n / EK-n (threshold = number of literals) -> every literal assigned true;
//   CARD-0 -> discarded;  EK-0 -> every literal assigned false.
// Readings where the paper is silent (B6): a literal repeated in a disjunction is kept once
// and a disjunction holding l and -l is discarded (tautology); a repeated variable in any other
// constraint is AFSAT_E_DUPLICATE (FE is multilinear only over distinct variables); contradictory prefix
// assignments, an at-least threshold above the length and an at-most threshold below 0 are
// AFSAT_E_UNSAT; an at-most threshold >= the length is trivially satisfied and discarded; after
// normalisation at-most-1 / exactly-1 / at-least-1 keep the library types ATMOST 1 / EXACTLY 1 / OR.
// Host only: nothing here touches a device.
#include <ctype.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>
#include <algorithm>
#include <new>
#include <string>
#include <vector>
#include "../../include/afsat.h"

struct afsat_problem {
    int32_t n_vars = 0;
    int32_t declared_vars = 0, declared_cons = 0;
    std::vector<int64_t> row_ptr{0};
    std::vector<int32_t> lit_var;
    std::vector<int8_t> lit_sign;
    std::vector<uint8_t> type;
    std::vector<int32_t> param;
    std::vector<int8_t> fixed;          // grown on demand; 0 free, -1 True, +1 False
    int64_t n_read = 0, n_units = 0, n_discarded = 0;
    std::string err;
};

namespace {

thread_local std::string g_parse_error;

struct Tok { const char *p; size_t n; int line; };

bool tok_is(const Tok &t, const char *s) { return strlen(s) == t.n && strncmp(t.p, s, t.n) == 0; }

// [+-]?digits, the whole token
bool tok_int(const Tok &t, long long *v)
{
    size_t i = 0;
    bool neg = false;
    if (i < t.n && (t.p[i] == '-' || t.p[i] == '+')) { neg = t.p[i] == '-'; ++i; }
    if (i >= t.n) return false;
    long long x = 0;
    for (; i < t.n; ++i) {
        if (!isdigit((unsigned char)t.p[i])) return false;
        x = x * 10 + (t.p[i] - '0');
        if (x > 2000000000LL) return false;
    }
    *v = neg ? -x : x;
    return true;
}

int fail(afsat_problem *P, int code, int line, const std::string &msg)
{
    char buf[64];
    snprintf(buf, sizeof buf, "line %d: ", line);
    P->err = std::string(buf) + msg;
    return code;
}

// prefix assignment "literal (var, sign) is TRUE"; sign +1: variable True (x = -1), -1: variable False (x = +1)
int assign(afsat_problem *P, int32_t var, int sign, bool lit_true, int line)
{
    const int8_t val = (int8_t)((sign > 0) == lit_true ? -1 : +1);
    if ((size_t)var >= P->fixed.size()) P->fixed.resize((size_t)var + 1, 0);
    if (P->fixed[var] != 0 && P->fixed[var] != val) return fail(P, AFSAT_E_UNSAT, line, "contradictory unit assignments");
    if (P->fixed[var] == 0) ++P->n_units;
    P->fixed[var] = val;
    return AFSAT_OK;
}

void emit(afsat_problem *P, int type, int param, const std::vector<int32_t> &vars, const std::vector<int8_t> &signs)
{
    for (size_t i = 0; i < vars.size(); ++i) { P->lit_var.push_back(vars[i]); P->lit_sign.push_back(signs[i]); }
    P->row_ptr.push_back((int64_t)P->lit_var.size());
    P->type.push_back((uint8_t)type);
    P->param.push_back(param);
}

// one constraint, already tokenised; type and threshold t already normalised to OR / XOR / NAE / ATLEAST t / ATMOST t / EXACTLY t
int add_constraint(afsat_problem *P, int type, long long t, std::vector<int32_t> &vars, std::vector<int8_t> &signs, int line)
{
    ++P->n_read;
    const int k0 = (int)vars.size();
    if (k0 == 0) return fail(P, AFSAT_E_LENGTH, line, "constraint without literals");
    // repeated variables
    if (type == AFSAT_OR) {
        std::vector<int32_t> v2; std::vector<int8_t> s2;
        for (int i = 0; i < k0; ++i) {
            bool dup = false;
            for (size_t j = 0; j < v2.size(); ++j)
                if (v2[j] == vars[i]) {
                    if (s2[j] != signs[i]) { ++P->n_discarded; return AFSAT_OK; }   // l or -l: tautology
                    dup = true;
                }
            if (!dup) { v2.push_back(vars[i]); s2.push_back(signs[i]); }
        }
        vars.swap(v2); signs.swap(s2);
    } else {
        for (int i = 0; i < k0; ++i)
            for (int j = 0; j < i; ++j)
                if (vars[i] == vars[j]) return fail(P, AFSAT_E_DUPLICATE, line, "variable repeated inside a constraint");
    }
    const int k = (int)vars.size();
    // the length limit binds only what reaches a kernel: constraints that A.1 turns into prefix assignments or discards
    // may be longer
    auto emit_c = [&](int ty, int prm) {
        if (k > AFSAT_MAX_LEN) return fail(P, AFSAT_E_LENGTH, line, "constraint longer than AFSAT_MAX_LEN");
        emit(P, ty, prm, vars, signs);
        return (int)AFSAT_OK;
    };
    auto all = [&](bool lit_true) {
        for (int i = 0; i < k; ++i) { int rc = assign(P, vars[i], signs[i], lit_true, line); if (rc) return rc; }
        return (int)AFSAT_OK;
    };
    switch (type) {
    case AFSAT_OR:
        if (k == 1) return all(true);                                  // unit CNF -> prefix assignment
        return emit_c(AFSAT_OR, 0);
    case AFSAT_XOR:
    case AFSAT_NAE:
        return emit_c(type, type == AFSAT_XOR ? 1 : 0);                // odd parity (Table 2)
    case AFSAT_ATLEAST:
        if (t <= 0) { ++P->n_discarded; return AFSAT_OK; }             // CARD-0: trivially satisfied
        if (t > k) return fail(P, AFSAT_E_UNSAT, line, "at-least threshold exceeds the number of literals");
        if (t == k) return all(true);                                  // CARD-n -> unit assignments
        if (t == 1) return emit_c(AFSAT_OR, 0);                        // CARD-1 -> CNF
        return emit_c(AFSAT_ATLEAST, (int)t);
    case AFSAT_ATMOST:
        if (t < 0) return fail(P, AFSAT_E_UNSAT, line, "at-most threshold below zero");
        if (t >= k) { ++P->n_discarded; return AFSAT_OK; }             // includes the unit AMO
        if (t == 0) return all(false);
        return emit_c(AFSAT_ATMOST, (int)t);
    case AFSAT_EXACTLY:
        if (t < 0 || t > k) return fail(P, AFSAT_E_UNSAT, line, "exactly-k with k outside [0, number of literals]");
        if (t == k) return all(true);                                  // EK-n, and the unit EO
        if (t == 0) return all(false);                                 // EK-0 -> negated assignments
        return emit_c(AFSAT_EXACTLY, (int)t);                          // EK-1 is EO = EXACTLY 1
    default:
        return fail(P, AFSAT_E_INVALID, line, "internal: unknown type");
    }
}

int parse_text(afsat_problem *P, const char *text, size_t len)
{
    // tokenise line by line: comment lines are dropped whole, everything else is one token stream
    std::vector<Tok> toks;
    int line = 1;
    size_t i = 0;
    while (i < len) {
        size_t e = i;
        while (e < len && text[e] != '\n') ++e;
        size_t s = i;
        while (s < e && isspace((unsigned char)text[s])) ++s;
        const bool comment = s < e && (text[s] == '*' || (text[s] == 'c' && (s + 1 == e || isspace((unsigned char)text[s + 1]))));
        if (!comment) {
            size_t q = s;
            while (q < e) {
                while (q < e && isspace((unsigned char)text[q])) ++q;
                size_t b = q;
                while (q < e && !isspace((unsigned char)text[q])) ++q;
                if (q > b) toks.push_back(Tok{text + b, q - b, line});
            }
        }
        i = e + 1;
        ++line;
    }
    size_t p = 0;
    std::vector<int32_t> vars;
    std::vector<int8_t> signs;
    while (p < toks.size()) {
        const int ln = toks[p].line;
        if (tok_is(toks[p], "p")) {                                    // p cnf V C
            long long V, Cc;
            if (p + 3 >= toks.size() || !tok_is(toks[p + 1], "cnf") || !tok_int(toks[p + 2], &V) || !tok_int(toks[p + 3], &Cc) || V < 1 || Cc < 0)
                return fail(P, AFSAT_E_INVALID, ln, "malformed problem line (expected: p cnf <vars> <constraints>)");
            P->declared_vars = std::max<int32_t>(P->declared_vars, (int32_t)V);
            P->declared_cons += (int32_t)Cc;
            p += 4;
            continue;
        }
        if (tok_is(toks[p], "h")) ++p;                                 // optional prefix
        if (p >= toks.size()) return fail(P, AFSAT_E_INVALID, ln, "dangling 'h'");
        int type = AFSAT_OR;
        long long t = 0;
        const Tok &id = toks[p];
        long long dummy;
        if (!tok_int(id, &dummy)) {
            ++p;
            if (tok_is(id, "x") || tok_is(id, "xor")) type = AFSAT_XOR;
            else if (tok_is(id, "n") || tok_is(id, "nae")) type = AFSAT_NAE;
            else if (tok_is(id, "a") || tok_is(id, "amo")) { type = AFSAT_ATMOST; t = 1; }
            else if (tok_is(id, "e") || tok_is(id, "eo")) { type = AFSAT_EXACTLY; t = 1; }
            else if (tok_is(id, "k") || tok_is(id, "ek")) {
                type = AFSAT_EXACTLY;
                if (p >= toks.size() || !tok_int(toks[p], &t)) return fail(P, AFSAT_E_INVALID, ln, "ek needs an integer count");
                ++p;
            } else if (tok_is(id, "d") || tok_is(id, "card")) {
                if (p >= toks.size()) return fail(P, AFSAT_E_INVALID, ln, "card needs a threshold");
                Tok th = toks[p++];
                int op = 0;                                            // 0 bare, 1 '<', 2 '<=', 3 '>', 4 '>='
                if (th.n >= 2 && th.p[0] == '<' && th.p[1] == '=') { op = 2; th.p += 2; th.n -= 2; }
                else if (th.n >= 2 && th.p[0] == '>' && th.p[1] == '=') { op = 4; th.p += 2; th.n -= 2; }
                else if (th.n >= 1 && th.p[0] == '<') { op = 1; th.p += 1; th.n -= 1; }
                else if (th.n >= 1 && th.p[0] == '>') { op = 3; th.p += 1; th.n -= 1; }
                if (op != 0 && th.n == 0) {                            // operator and number as two tokens
                    if (p >= toks.size()) return fail(P, AFSAT_E_INVALID, ln, "card needs a threshold");
                    th = toks[p++];
                }
                long long kk;
                if (!tok_int(th, &kk)) return fail(P, AFSAT_E_INVALID, ln, "card threshold is not an integer");
                if (op != 0 && kk < 1) return fail(P, AFSAT_E_INVALID, ln, "card threshold after an operator must be positive");
                if (op == 0 && kk == 0) return fail(P, AFSAT_E_INVALID, ln, "card threshold 0 terminates nothing");
                if (op == 0) { if (kk > 0) { type = AFSAT_ATLEAST; t = kk; } else { type = AFSAT_ATMOST; t = -kk - 1; } }
                else if (op == 1) { type = AFSAT_ATMOST; t = kk - 1; }
                else if (op == 2) { type = AFSAT_ATMOST; t = kk; }
                else if (op == 3) { type = AFSAT_ATLEAST; t = kk + 1; }
                else { type = AFSAT_ATLEAST; t = kk; }
            } else {
                return fail(P, AFSAT_E_INVALID, ln, "unknown constraint identifier '" + std::string(id.p, id.n) + "'");
            }
        }
        vars.clear(); signs.clear();
        bool closed = false;
        while (p < toks.size()) {
            long long l;
            if (!tok_int(toks[p], &l)) return fail(P, AFSAT_E_INVALID, toks[p].line, "expected a literal, got '" + std::string(toks[p].p, toks[p].n) + "'");
            ++p;
            if (l == 0) { closed = true; break; }
            const long long v = l < 0 ? -l : l;
            if (v > AFSAT_PARSE_MAX_VARS) return fail(P, AFSAT_E_VARIABLE, ln, "variable index too large");
            vars.push_back((int32_t)(v - 1));
            signs.push_back((int8_t)(l > 0 ? +1 : -1));
            P->n_vars = std::max<int32_t>(P->n_vars, (int32_t)v);
        }
        if (!closed) return fail(P, AFSAT_E_INVALID, ln, "constraint not terminated by 0");
        const int end_line = toks[p - 1].line;                        // trailing comment on the closing line
        if (p < toks.size() && toks[p].line == end_line && (tok_is(toks[p], "c") || toks[p].p[0] == '*'))
            while (p < toks.size() && toks[p].line == end_line) ++p;
        int rc = add_constraint(P, type, t, vars, signs, ln);
        if (rc) return rc;
    }
    P->n_vars = std::max(P->n_vars, P->declared_vars);
    if (P->n_vars < 1) return fail(P, AFSAT_E_INVALID, line, "no variables");
    P->fixed.resize((size_t)P->n_vars, 0);
    return AFSAT_OK;
}

}  // namespace

extern "C" {

int afsat_parse(const char *text, int64_t len, afsat_problem **out)
{
    if (!out || !text || len < 0) { g_parse_error = "afsat_parse: NULL pointer or negative length"; return AFSAT_E_INVALID; }
    *out = nullptr;
    afsat_problem *P = new (std::nothrow) afsat_problem();
    if (!P) { g_parse_error = "out of host memory"; return AFSAT_E_NOMEM; }
    int rc = parse_text(P, text, (size_t)len);
    if (rc) { g_parse_error = P->err; delete P; return rc; }
    *out = P;
    return AFSAT_OK;
}

int afsat_parse_file(const char *path, afsat_problem **out)
{
    if (!out || !path) { g_parse_error = "afsat_parse_file: NULL pointer"; return AFSAT_E_INVALID; }
    *out = nullptr;
    FILE *f = fopen(path, "rb");
    if (!f) { g_parse_error = std::string("cannot open ") + path; return AFSAT_E_INVALID; }
    std::string buf;
    char tmp[1 << 16];
    size_t r;
    while ((r = fread(tmp, 1, sizeof tmp, f)) > 0) buf.append(tmp, r);
    fclose(f);
    return afsat_parse(buf.data(), (int64_t)buf.size(), out);
}

const char *afsat_parse_error(void) { return g_parse_error.c_str(); }

int afsat_problem_sizes(const afsat_problem *P, int32_t *n_vars, int32_t *n_cons, int64_t *nnz, int64_t *stats)
{
    if (!P) return AFSAT_E_INVALID;
    if (n_vars) *n_vars = P->n_vars;
    if (n_cons) *n_cons = (int32_t)P->type.size();
    if (nnz) *nnz = (int64_t)P->lit_var.size();
    if (stats) {
        stats[0] = P->n_read; stats[1] = P->n_units; stats[2] = P->n_discarded;
        stats[3] = P->declared_vars; stats[4] = P->declared_cons;
    }
    return AFSAT_OK;
}

int afsat_problem_fill(const afsat_problem *P, int64_t *row_ptr, int32_t *lit_var, int8_t *lit_sign, uint8_t *type,
                       int32_t *param, int8_t *fixed)
{
    if (!P || !row_ptr || !fixed) return AFSAT_E_INVALID;
    const size_t m = P->type.size(), nnz = P->lit_var.size();
    if ((m && (!type || !param)) || (nnz && (!lit_var || !lit_sign))) return AFSAT_E_INVALID;
    memcpy(row_ptr, P->row_ptr.data(), (m + 1) * sizeof(int64_t));
    if (nnz) { memcpy(lit_var, P->lit_var.data(), nnz * sizeof(int32_t)); memcpy(lit_sign, P->lit_sign.data(), nnz); }
    if (m) { memcpy(type, P->type.data(), m); memcpy(param, P->param.data(), m * sizeof(int32_t)); }
    memcpy(fixed, P->fixed.data(), (size_t)P->n_vars);
    return AFSAT_OK;
}

void afsat_problem_free(afsat_problem *P) { delete P; }

}  // extern "C"
