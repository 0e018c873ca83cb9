/* Fast Jordan-Wigner builder for the synthetic workloads (input GENERATOR, not the method).
 *
 * H = sum_{pq,s} h_pq a+_{ps} a_{qs} + 1/2 sum_{pqrs,s,t} g_pqrs a+_{ps} a+_{rt} a_{st} a_{qs}
 * with g_pqrs = (pq|rs) (chemists' notation), spin-orbital index j = 2p + s (alpha even, beta odd;
 * PAPER.md:116-118 Eq. 12) and the OpenFermion convention
 *   a_j  = (prod_{k<j} Z_k) (X_j + iY_j)/2,   a+_j = (prod_{k<j} Z_k) (X_j - iY_j)/2.
 *
 * Operators are kept as real-weighted monomials X^x Z^z (x, z: 128-bit masks); since
 * X_j + iY_j = X_j (1 - Z_j) and X_j - iY_j = X_j (1 + Z_j) every ladder operator is two
 * monomials with weights +-1/2 and every product stays real.  A monomial with ny = |x & z|
 * doubly-set positions equals (-i)^ny times the Pauli string that has Y there, so the Pauli
 * coefficient is c * (-i)^ny; for a Hermitian H with real integrals the odd-ny parts cancel
 * (their largest residual is reported so the caller can assert it).
 *
 * Output: Pauli strings as (x, z) mask pairs, x = X-or-Y positions, z = Y-or-Z positions
 * (2 x uint64, qubit j <-> bit j%64 of word j/64), real coefficients, |c| < tol dropped,
 * identity kept.  Order = hash-table order (deterministic function of the inputs, deliberately
 * unsorted so that a Hamiltonian compiler downstream has real work to do).
 *
 * Build: gcc -O2 -shared -fPIC jwgen.c -o _jwgen.so
 */
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#include <math.h>

typedef struct { uint64_t x[2], z[2]; double c; } mono_t;
typedef struct { uint64_t x[2], z[2]; double c; int used; } slot_t;

static inline int par2(uint64_t a0, uint64_t a1) {
    return (__builtin_popcountll(a0) + __builtin_popcountll(a1)) & 1;
}

static inline mono_t mmul(const mono_t *a, const mono_t *b) {
    mono_t r;
    int sg = par2(a->z[0] & b->x[0], a->z[1] & b->x[1]);   /* Z^z1 X^x2 = (-1)^{z1.x2} X^x2 Z^z1 */
    r.x[0] = a->x[0] ^ b->x[0]; r.x[1] = a->x[1] ^ b->x[1];
    r.z[0] = a->z[0] ^ b->z[0]; r.z[1] = a->z[1] ^ b->z[1];
    r.c = sg ? -(a->c * b->c) : (a->c * b->c);
    return r;
}

static void ladder(int j, int dagger, mono_t out[2]) {
    uint64_t e[2] = {0, 0}, m[2] = {0, 0};
    e[j >> 6] = 1ull << (j & 63);
    if (j >= 64) { m[0] = ~0ull; m[1] = (1ull << (j - 64)) - 1; }      /* Z string on qubits < j */
    else         { m[0] = (1ull << j) - 1; }
    out[0].x[0] = e[0]; out[0].x[1] = e[1]; out[0].z[0] = m[0];        out[0].z[1] = m[1];        out[0].c = 0.5;
    out[1].x[0] = e[0]; out[1].x[1] = e[1]; out[1].z[0] = m[0] | e[0]; out[1].z[1] = m[1] | e[1]; out[1].c = dagger ? 0.5 : -0.5;
}

static inline uint64_t mix(uint64_t h) {
    h ^= h >> 33; h *= 0xff51afd7ed558ccdull; h ^= h >> 33; h *= 0xc4ceb9fe1a85ec53ull; h ^= h >> 33;
    return h;
}

typedef struct { slot_t *t; uint64_t mask; int64_t n; } table_t;

static int tadd(table_t *T, const mono_t *m, double scale) {
    uint64_t h = mix(m->x[0] ^ mix(m->x[1] + 0x9e3779b97f4a7c15ull) ^ mix(m->z[0] * 3 + 1) ^ mix(m->z[1] * 7 + 5));
    uint64_t i = h & T->mask;
    for (;;) {
        slot_t *s = &T->t[i];
        if (!s->used) {
            if ((uint64_t)T->n * 10 > (T->mask + 1) * 7) return -1;      /* load > 0.7: caller retries bigger */
            s->used = 1; s->x[0] = m->x[0]; s->x[1] = m->x[1]; s->z[0] = m->z[0]; s->z[1] = m->z[1];
            s->c = m->c * scale; T->n++;
            return 0;
        }
        if (s->x[0] == m->x[0] && s->x[1] == m->x[1] && s->z[0] == m->z[0] && s->z[1] == m->z[1]) {
            s->c += m->c * scale;
            return 0;
        }
        i = (i + 1) & T->mask;
    }
}

/* Returns the number of terms written (<= max_terms), -1 if the table (2^cap_log2 slots) or the
 * output buffers were too small, -2 on allocation failure.  *max_imag receives the largest
 * |coefficient| found on an odd-Y (would-be imaginary) string before it was discarded. */
int64_t jw_build(int n_spatial, const double *h, const double *g, double tol, int cap_log2,
                 int64_t max_terms, uint64_t *out_x, uint64_t *out_z, double *out_c, double *max_imag)
{
    const int N = n_spatial, n = 2 * N;
    if (n > 128 || n < 1) return -1;
    table_t T; T.mask = (1ull << cap_log2) - 1; T.n = 0;
    T.t = (slot_t *)calloc((size_t)1 << cap_log2, sizeof(slot_t));
    if (!T.t) return -2;

    mono_t (*cr)[2] = malloc(sizeof(mono_t[2]) * n), (*an)[2] = malloc(sizeof(mono_t[2]) * n);
    for (int j = 0; j < n; ++j) { ladder(j, 1, cr[j]); ladder(j, 0, an[j]); }
    int fail = 0;

    /* one-body */
    for (int p = 0; p < N && !fail; ++p) for (int q = 0; q < N && !fail; ++q) {
        double hv = h[p * N + q];
        if (hv == 0.0) continue;
        for (int s = 0; s < 2; ++s) {
            int j1 = 2 * p + s, j2 = 2 * q + s;
            for (int a = 0; a < 2; ++a) for (int b = 0; b < 2; ++b) {
                mono_t m = mmul(&cr[j1][a], &an[j2][b]);
                if (tadd(&T, &m, hv)) fail = 1;
            }
        }
    }
    /* two-body: 1/2 g_pqrs a+_{ps} a+_{rt} a_{st} a_{qs} */
    for (int p = 0; p < N && !fail; ++p) for (int q = 0; q < N && !fail; ++q)
    for (int r = 0; r < N && !fail; ++r) for (int s4 = 0; s4 < N && !fail; ++s4) {
        double gv = g[((p * N + q) * N + r) * N + s4];
        if (gv == 0.0) continue;
        for (int s = 0; s < 2; ++s) for (int t = 0; t < 2; ++t) {
            int j1 = 2 * p + s, j2 = 2 * r + t, j3 = 2 * s4 + t, j4 = 2 * q + s;
            if (j1 == j2 || j3 == j4) continue;                       /* a+a+ = aa = 0 on equal modes */
            for (int a = 0; a < 2; ++a) for (int b = 0; b < 2; ++b) {
                mono_t m12 = mmul(&cr[j1][a], &cr[j2][b]);
                for (int c = 0; c < 2; ++c) for (int d = 0; d < 2; ++d) {
                    mono_t m34 = mmul(&an[j3][c], &an[j4][d]);
                    mono_t m = mmul(&m12, &m34);
                    if (tadd(&T, &m, 0.5 * gv)) fail = 1;
                }
            }
        }
    }
    free(cr); free(an);
    if (fail) { free(T.t); return -1; }

    int64_t k = 0; double mi = 0.0;
    for (uint64_t i = 0; i <= T.mask; ++i) {
        slot_t *s = &T.t[i];
        if (!s->used) continue;
        int ny = __builtin_popcountll(s->x[0] & s->z[0]) + __builtin_popcountll(s->x[1] & s->z[1]);
        if (ny & 1) { if (fabs(s->c) > mi) mi = fabs(s->c); continue; }
        double c = (ny & 2) ? -s->c : s->c;                            /* (-i)^ny, ny even */
        if (fabs(c) < tol) continue;
        if (k >= max_terms) { free(T.t); return -1; }
        out_x[2 * k] = s->x[0]; out_x[2 * k + 1] = s->x[1];
        out_z[2 * k] = s->z[0]; out_z[2 * k + 1] = s->z[1];
        out_c[k] = c; ++k;
    }
    free(T.t);
    if (max_imag) *max_imag = mi;
    return k;
}
