// (a1) Hamiltonian compiler — host only.  PAPER.md:154-156: parse the Operator Matrix into incidence rows
// F^{1,2} (flips) / F^{2,3} (signs), keep a buffer of unique flips and their number of occurrences.
// Rules 1-5 are stated in include/nqs.h.
#include <algorithm>
#include <charconv>
#include <cmath>
#include <system_error>
#include <new>
#include <numeric>
#include <cstdlib>
#include <string>
#include "nqs_internal.h"

namespace {

struct Term { uint64_t f[2], s[2]; int64_t idx; };

inline bool key_less(const Term &a, const Term &b) {
    if (a.f[1] != b.f[1]) return a.f[1] < b.f[1];
    if (a.f[0] != b.f[0]) return a.f[0] < b.f[0];
    if (a.s[1] != b.s[1]) return a.s[1] < b.s[1];
    return a.s[0] < b.s[0];
}
inline bool key_eq(const Term &a, const Term &b) {
    return a.f[0] == b.f[0] && a.f[1] == b.f[1] && a.s[0] == b.s[0] && a.s[1] == b.s[1];
}

int finish(int n, std::vector<Term> &terms, const double *coeffs, nqs_ham_t **out) {
    // stable sort keeps input order among identical strings -> left-to-right fp64 merge (rule 2)
    std::stable_sort(terms.begin(), terms.end(), key_less);
    nqs_ham *H = new (std::nothrow) nqs_ham();
    if (!H) return NQS_ENOMEM;
    H->n = n;
    try {
        const size_t T = terms.size();
        size_t i = 0;
        bool have_group = false;
        uint64_t gf[2] = {0, 0};
        while (i < T) {
            size_t j = i;
            double c = coeffs[terms[i].idx];
            for (j = i + 1; j < T && key_eq(terms[j], terms[i]); ++j) c = c + coeffs[terms[j].idx];
            if (c != 0.0) {                                                      // rule 3
                const Term &t = terms[i];
                if (!have_group || gf[0] != t.f[0] || gf[1] != t.f[1]) {
                    H->flips.push_back(t.f[0]); H->flips.push_back(t.f[1]);
                    H->offsets.push_back((uint32_t)H->coef.size());
                    gf[0] = t.f[0]; gf[1] = t.f[1]; have_group = true;
                }
                H->zy.push_back(t.s[0]); H->zy.push_back(t.s[1]);
                H->ycount.push_back((uint8_t)(__builtin_popcountll(t.f[0] & t.s[0]) +
                                              __builtin_popcountll(t.f[1] & t.s[1])));
                H->coef.push_back((float)c);                                     // RNE (rule 5)
                H->sum_abs += std::fabs(c);
            }
            i = j;
        }
        H->offsets.push_back((uint32_t)H->coef.size());
        H->K = (int64_t)H->coef.size();
        H->G = (int64_t)H->offsets.size() - 1;
    } catch (const std::bad_alloc &) {
        delete H;
        return NQS_ENOMEM;
    }
    *out = H;
    return NQS_OK;
}

inline bool high_bits_clear(int n, const uint64_t m[2]) {
    if (n >= 128) return true;
    if (n >= 64) return (n == 64 ? m[1] == 0 : (m[1] >> (n - 64)) == 0);
    return m[1] == 0 && (m[0] >> n) == 0;
}

}  // namespace

extern "C" int nqs_ham_compile(int n_qubits, int64_t n_terms, const uint8_t *codes, const double *coeffs,
                               nqs_ham_t **out) {
    if (!out || n_terms < 0 || (n_terms > 0 && (!codes || !coeffs))) return NQS_EINVAL;
    if (n_qubits < 3 || n_qubits > NQS_MAX_QUBITS) return NQS_ERANGE;
    if (n_terms > 0xFFFFFFF0ll) return NQS_ERANGE;
    std::vector<Term> terms;
    try { terms.resize((size_t)n_terms); } catch (const std::bad_alloc &) { return NQS_ENOMEM; }
    for (int64_t k = 0; k < n_terms; ++k) {
        Term t{{0, 0}, {0, 0}, k};
        const uint8_t *row = codes + (size_t)k * n_qubits;
        for (int j = 0; j < n_qubits; ++j) {
            const uint8_t p = row[j];
            if (p > 3) return NQS_EINVAL;
            const uint64_t bit = 1ull << (j & 63);
            if (p == 1 || p == 2) t.f[j >> 6] |= bit;       // sigma_1, sigma_2 flip  (F^{1,2})
            if (p == 2 || p == 3) t.s[j >> 6] |= bit;       // sigma_2, sigma_3 sign  (F^{2,3})
        }
        terms[(size_t)k] = t;
    }
    return finish(n_qubits, terms, coeffs, out);
}

extern "C" int nqs_ham_compile_packed(int n_qubits, int64_t n_terms, const uint64_t *fmask,
                                      const uint64_t *smask, const double *coeffs, nqs_ham_t **out) {
    if (!out || n_terms < 0 || (n_terms > 0 && (!fmask || !smask || !coeffs))) return NQS_EINVAL;
    if (n_qubits < 3 || n_qubits > NQS_MAX_QUBITS) return NQS_ERANGE;
    if (n_terms > 0xFFFFFFF0ll) return NQS_ERANGE;
    std::vector<Term> terms;
    try { terms.resize((size_t)n_terms); } catch (const std::bad_alloc &) { return NQS_ENOMEM; }
    for (int64_t k = 0; k < n_terms; ++k) {
        Term t{{fmask[2 * k], fmask[2 * k + 1]}, {smask[2 * k], smask[2 * k + 1]}, k};
        if (!high_bits_clear(n_qubits, t.f) || !high_bits_clear(n_qubits, t.s)) return NQS_EINVAL;
        terms[(size_t)k] = t;
    }
    return finish(n_qubits, terms, coeffs, out);
}

// [sign] digits [. digits] [e [sign] digits] -> finite double; *end = first character after it.
static bool parse_decimal(const char *first, const char *last, double *value, const char **end) {
    const char *p = first;
    if (p < last && (*p == '+' || *p == '-')) ++p;
    if (p >= last || !((*p >= '0' && *p <= '9') || *p == '.')) return false;          // no "nan", "inf", "x..."
    const std::from_chars_result r = std::from_chars(*first == '+' ? first + 1 : first, last, *value, std::chars_format::general);
    if (r.ec != std::errc() || !std::isfinite(*value)) return false;                   // overflow ("1e400") included
    *end = r.ptr;
    return true;
}

// Text form of a qubit Hamiltonian (PAPER.md:36 "stored in a string format", :154 "string parser"; the syntax is not
// given, reading A4): one term per line, coefficient first, then EITHER a dense word of n_qubits letters from IXYZ
// (letter j = qubit j) OR sparse factors "X0 Y3 Z12" (identity = nothing).  The coefficient may be written plainly
// ("-0.25"), in parentheses, or as a complex literal with a zero imaginary part ("(0.5+0j)", the OpenFermion print
// form); '[' ']' '*' ',' are separators; '#' starts a comment.
extern "C" int nqs_ham_compile_text(int n_qubits, const char *text, nqs_ham_t **out) {
    if (!out || !text) return NQS_EINVAL;
    if (n_qubits < 3 || n_qubits > NQS_MAX_QUBITS) return NQS_ERANGE;
    std::vector<Term> terms;
    std::vector<double> coeffs;
    try {
        const char *p = text;
        while (*p) {
            const char *eol = p;
            while (*eol && *eol != '\n') ++eol;
            std::string line(p, eol);
            p = *eol ? eol + 1 : eol;
            const size_t hash = line.find('#');
            if (hash != std::string::npos) line.resize(hash);
            for (char &ch : line) if (ch == '[' || ch == ']' || ch == '*' || ch == ',' || ch == '(' || ch == ')' || ch == '\t' || ch == '\r') ch = ' ';
            size_t i = line.find_first_not_of(' ');
            if (i == std::string::npos) continue;
            // decimal, finite, locale-independent: std::from_chars never reads hex ("0X1 Z2" is 0 * X1 Z2 mangled,
            // not 1.0 * Z2) and "nan" / "inf" / overflowing literals are refused so that sum|c| stays a number
            const char *end = nullptr;
            double c = 0.0;
            if (!parse_decimal(line.c_str() + i, line.c_str() + line.size(), &c, &end)) return NQS_EINVAL;
            // optional imaginary part "+0j" / "-0.0j": must be zero (real coefficients)
            if (*end == '+' || *end == '-') {
                const char *e2 = nullptr;
                double im = 0.0;
                if (parse_decimal(end, line.c_str() + line.size(), &im, &e2) && (*e2 == 'j' || *e2 == 'i')) {
                    if (im != 0.0) return NQS_EINVAL;
                    end = e2 + 1;
                }
            }
            if (*end && *end != ' ') return NQS_EINVAL;                       // the coefficient is a token of its own
            uint64_t named[2] = {0, 0};                                       // qubits this line has named, I included
            Term t{{0, 0}, {0, 0}, (int64_t)terms.size()};
            const char *q = end;
            bool dense_seen = false;
            while (*q) {
                while (*q == ' ') ++q;
                if (!*q) break;
                const char *w = q;
                while (*q && *q != ' ') ++q;
                const size_t len = (size_t)(q - w);
                auto put = [&](char letter, int j) -> bool {
                    if (j < 0 || j >= n_qubits) return false;
                    const uint64_t bit = 1ull << (j & 63);
                    if (named[j >> 6] & bit) return false;                        // qubit named twice, in either order
                    named[j >> 6] |= bit;
                    switch (letter) {
                        case 'I': return true;
                        case 'X': t.f[j >> 6] |= bit; return true;
                        case 'Y': t.f[j >> 6] |= bit; t.s[j >> 6] |= bit; return true;
                        case 'Z': t.s[j >> 6] |= bit; return true;
                        default: return false;
                    }
                };
                bool all_letters = true;
                for (size_t k = 0; k < len; ++k) if (!(w[k] == 'I' || w[k] == 'X' || w[k] == 'Y' || w[k] == 'Z')) all_letters = false;
                if (all_letters && (int)len == n_qubits && !dense_seen) {
                    for (int j = 0; j < n_qubits; ++j) if (!put(w[j], j)) return NQS_EINVAL;
                    dense_seen = true;
                } else if (len >= 2 && (w[0] == 'X' || w[0] == 'Y' || w[0] == 'Z' || w[0] == 'I')) {
                    char *e3 = nullptr;
                    const long j = strtol(w + 1, &e3, 10);
                    if (e3 != q || !put(w[0], (int)j)) return NQS_EINVAL;
                } else {
                    return NQS_EINVAL;
                }
            }
            terms.push_back(t);
            coeffs.push_back(c);
        }
    } catch (const std::bad_alloc &) { return NQS_ENOMEM; }
    if (terms.size() > 0xFFFFFFF0ull) return NQS_ERANGE;
    return finish(n_qubits, terms, coeffs.data(), out);
}

extern "C" int nqs_ham_info(const nqs_ham_t *ham, int *n_qubits, int64_t *K, int64_t *G, double *sum_abs_coeff) {
    if (!ham) return NQS_EINVAL;
    if (n_qubits) *n_qubits = ham->n;
    if (K) *K = ham->K;
    if (G) *G = ham->G;
    if (sum_abs_coeff) *sum_abs_coeff = ham->sum_abs;
    return NQS_OK;
}

extern "C" int nqs_ham_export(const nqs_ham_t *ham, uint64_t *flips, uint32_t *offsets, uint64_t *zy,
                              uint8_t *ycount, float *coef) {
    if (!ham) return NQS_EINVAL;
    if (flips)   std::copy(ham->flips.begin(), ham->flips.end(), flips);
    if (offsets) std::copy(ham->offsets.begin(), ham->offsets.end(), offsets);
    if (zy)      std::copy(ham->zy.begin(), ham->zy.end(), zy);
    if (ycount)  std::copy(ham->ycount.begin(), ham->ycount.end(), ycount);
    if (coef)    std::copy(ham->coef.begin(), ham->coef.end(), coef);
    return NQS_OK;
}
