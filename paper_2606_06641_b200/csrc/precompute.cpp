// precompute.cpp -- host-side, once per signature (type, k, param): SURVEY.md §8(a) step a0.
//
// Builds what the kernels contract the DFT-point products with (§2.1.2) following
// the "tailored DFT construction" of PAPER.md:141-147 (§3.5.1):
//   * the Fourier coefficients are EXACT INTEGERS A_j = 2^k f^(S), |S| = j, obtained from the
//     generating polynomial (1-u)^j (1+u)^(k-j) in 128-bit integer arithmetic ("arbitrary
//     precision integer arithmetic, division deferred");
//   * roots of unity are never produced by repeated multiplication: each w^(l j)
//     is looked up by its reduced exponent (l j mod N) and evaluated after an exact integer
//     reduction of the angle to the first octant, so that w^(N-l) == conj(w^l) bit for bit,
//     w^0 = 1, w^(N/2) = -1, w^(N/4) = i exactly ("explicitly mirrored");
//   * sums are taken in IEEE binary128 and the only division (by N; the 2^k is folded into the
//     factors as an exact power of two) happens last.
// With P_l(y) = prod_i (1 + w^l y_i)/2  (the paper's product, each factor halved -- an exact
// power-of-two rescale, reading A7) the result is
//     FE(y) = sum_{l<H} Re( w_l P_l ),   w_l = (c_l / N) sum_j A_j w^(-l j),
// c_l = 1 for the self-conjugate points l = 0 and l = N/2, else 2 (points l > N/2 are the complex
// conjugates and are never evaluated), N = k+1, H = floor(N/2)+1.
//
// This file shares no code with the CPU test oracle (which uses Krawtchouk sums and no DFT).
#include <quadmath.h>
#include <string.h>
#include <vector>
#include "afsat_internal.h"

typedef __float128 Q;
typedef __int128 I128;

bool afsat_sig_satisfied(int32_t type, int32_t k, int32_t param, int32_t tau)
{
    switch (type) {
    case AFSAT_OR:      return tau > 0;
    case AFSAT_XOR:     return ((tau ^ param) & 1) == 0;
    case AFSAT_ATLEAST: return tau >= param;
    case AFSAT_ATMOST:  return tau <= param;
    case AFSAT_EXACTLY: return tau == param;
    case AFSAT_NAE:     return tau != 0 && tau != k;
    default:            return false;
    }
}

// exp(2 pi i num/den), 0 <= num < den, with exact symmetries (see header comment).
static void unit_root(long num, long den, Q *c, Q *s)
{
    bool conj = false, negc = false, swp = false;
    if (2 * num > den) { num = den - num; conj = true; }              // lower half: mirror
    if (4 * num > den) { num = den - 2 * num; den *= 2; negc = true; } // 2nd quadrant: pi - theta
    if (8 * num > den) { num = den - 4 * num; den *= 4; swp = true; }  // 2nd octant: pi/2 - theta
    Q ang = 2 * M_PIq * (Q)num / (Q)den;                              // now in [0, pi/4]
    Q cc = cosq(ang), ss = sinq(ang);
    if (num == 0) { cc = 1; ss = 0; }
    if (swp) { Q t = cc; cc = ss; ss = t; }
    if (negc) cc = -cc;
    if (conj) ss = -ss;
    *c = cc; *s = ss;
}

// [u^tau] (1-u)^j (1+u)^(k-j), tau = 0..k, exact.
static void char_poly(int k, int j, I128 *poly)
{
    for (int t = 0; t <= k; ++t) poly[t] = 0;
    poly[0] = 1;
    int deg = 0;
    for (int r = 0; r < k; ++r) {
        int sgn = (r < j) ? -1 : +1;                                   // times (1 -+ u)
        for (int t = deg + 1; t >= 1; --t) poly[t] += sgn * poly[t - 1];
        ++deg;
    }
}

int afsat_sig_build(int32_t type, int32_t k, int32_t param, uint32_t flags, AfsatSigHost *out)
{
    if (!out) return AFSAT_E_INVALID;
    if (type < AFSAT_OR || type > AFSAT_NAE) return AFSAT_E_INVALID;
    if (k < 1 || k > AFSAT_MAX_LEN) return AFSAT_E_LENGTH;
    if (type == AFSAT_XOR && param != 0 && param != 1) return AFSAT_E_PARAM;
    if ((type == AFSAT_ATLEAST || type == AFSAT_ATMOST || type == AFSAT_EXACTLY) &&
        (param < 0 || param > k))
        return AFSAT_E_PARAM;
    uint64_t lo = 0, hi = 0;
    for (int tau = 0; tau <= k; ++tau)
        if (afsat_sig_satisfied(type, k, param, tau)) { if (tau < 64) lo |= 1ull << tau; else hi |= 1ull << (tau - 64); }
    int rc = afsat_sig_build_mask(k, lo, hi, flags, out);
    if (rc) return rc;
    out->type = type; out->param = (type == AFSAT_OR || type == AFSAT_NAE) ? 0 : param;
    return AFSAT_OK;
}

// The same for ANY symmetric constraint on k literals, given as the set of satisfying counts (bit tau of the mask):
// what a Table 1 constraint becomes once a partial assignment has decided some of its literals.
int afsat_sig_build_mask(int32_t k, uint64_t satmask_lo, uint64_t satmask_hi, uint32_t flags, AfsatSigHost *out)
{
    if (!out) return AFSAT_E_INVALID;
    if (k < 1 || k > AFSAT_MAX_LEN) return AFSAT_E_LENGTH;
    memset(out, 0, sizeof *out);
    out->type = -1; out->k = k; out->param = 0;
    out->satmask_lo = satmask_lo; out->satmask_hi = satmask_hi;
    const int N = k + 1, H = N / 2 + 1;
    const bool robust = (flags & AFSAT_FLAG_ROBUST) != 0;

    int g[AFSAT_MAX_LEN + 1];                                          // +-1 truth table
    for (int tau = 0; tau <= k; ++tau) {
        const bool sat = ((tau < 64 ? satmask_lo >> tau : satmask_hi >> (tau - 64)) & 1ull) != 0;
        g[tau] = sat ? -1 : +1;
    }

    // the spectrum that multiplies the products: integer sequence s_j and its scale
    I128 seq[AFSAT_MAX_LEN + 1];
    Q seq_abs_sum = 0;
    if (!robust) {
        I128 poly[AFSAT_MAX_LEN + 1];
        for (int j = 0; j <= k; ++j) {                                 // A_j = sum_tau g(tau) K_tau(j)
            char_poly(k, j, poly);
            I128 a = 0;
            for (int tau = 0; tau <= k; ++tau) a += g[tau] * poly[tau];
            seq[j] = a;
        }
    } else {
        for (int j = 0; j <= k; ++j) seq[j] = g[j];                    // robust: DFT of g itself
    }
    for (int j = 0; j <= k; ++j) seq_abs_sum += (Q)(seq[j] < 0 ? -seq[j] : seq[j]);

    struct Pt { Q ar, ai, br, bi, wr, wi; bool real; };
    std::vector<Pt> pts;
    for (int l = 0; l < H; ++l) {
        Q sr = 0, si = 0;                                              // sum_j s_j w^(-l j)
        for (int j = 0; j <= k; ++j) {
            long e = (long)(((long)l * j) % N);
            Q c, s;
            unit_root((N - e) % N, N, &c, &s);
            sr += (Q)seq[j] * c;
            si += (Q)seq[j] * s;
        }
        const bool self_conj = (l == 0) || (2 * l == N);
        if (self_conj) si = 0;
        if (fabsq(sr) + fabsq(si) <= seq_abs_sum * 0x1p-80Q) continue; // exactly-zero weight: skip
        Q cl = self_conj ? 1 : 2;
        Pt p;
        p.wr = cl * sr / (Q)N;                                          // the single division
        p.wi = cl * si / (Q)N;
        Q c, s;
        unit_root(l, N, &c, &s);
        if (!robust) { p.ar = 0.5Q; p.ai = 0; p.br = c / 2; p.bi = s / 2; }
        else { p.ar = (1 + c) / 2; p.ai = s / 2; p.br = (1 - c) / 2; p.bi = -s / 2; }
        p.real = self_conj;
        pts.push_back(p);
    }
    int row = 0;
    for (int pass = 0; pass < 2; ++pass) {
        for (const Pt &p : pts) {
            if (p.real != (pass == 0)) continue;
            double *r = out->rows + 8 * row++;
            Q wbr = p.wr * p.br - p.wi * p.bi, wbi = p.wr * p.bi + p.wi * p.br;
            r[0] = (double)p.ar; r[1] = (double)p.ai; r[2] = (double)p.br; r[3] = (double)p.bi;
            r[4] = (double)p.wr; r[5] = (double)p.wi; r[6] = (double)wbr;  r[7] = (double)wbi;
            if (p.real) { r[1] = r[3] = r[5] = r[7] = 0.0; ++out->n_real; } else ++out->n_cplx;
        }
    }
    return AFSAT_OK;
}
