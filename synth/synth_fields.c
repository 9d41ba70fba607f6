/*
 * synth_fields.c -- seeded synthetic input generators (SURVEY.md 8(c) reading A20).
 *
 * This module feeds BOTH the oracle and the CUDA path with identical host
 * arrays; it holds none of the method's arithmetic (no shift, plaquette,
 * staple, projection, hop or reduction).  It stands in for the paper's
 * dynamical gauge configurations (beta=5.20 / 5.29), which
 * are not available: the shapes, sizes and value distributions are those of
 * BASELINE.json:configs.
 *
 * Every value is a pure function of (seed, field_id, element counter), so the
 * result does not depend on traversal order or thread count:
 *   counter -> SplitMix64 finaliser -> two uniforms -> Box-Muller normal pair.
 *
 *   hot  links: 3x3 complex i.i.d. N(0,1); Gram-Schmidt on rows 0,1;
 *               row 2 = conj(row0 x row1)          (Haar-like SU(3))
 *   warm links: A i.i.d. complex N(0,1); H = (A + A^dag)/2 - tr/3;
 *               U = exp(i eps H) by scaling-and-squaring Taylor series
 *   spinors   : 12 complex per site, i.i.d. N(0,1) real and imaginary parts
 *
 * Host layout: lexicographic sites, site-outermost (see include/qdp_b200.h).
 */
#include <math.h>
#include <stddef.h>
#include <stdint.h>
#include <string.h>

static uint64_t mix64(uint64_t z) {
    z += 0x9E3779B97F4A7C15ULL;
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
    return z ^ (z >> 31);
}
static uint64_t stream_key(uint64_t seed, uint64_t field_id) {
    return mix64(mix64(seed) ^ (field_id * 0xD6E8FEB86659FD93ULL));
}
static double u01(uint64_t r) { return ((double)(r >> 11) + 0.5) * (1.0 / 9007199254740992.0); }

/* normal pair number `ctr` of stream `key` */
static void normal_pair(uint64_t key, uint64_t ctr, double *a, double *b) {
    uint64_t r1 = mix64(key ^ mix64(2 * ctr));
    uint64_t r2 = mix64(key ^ mix64(2 * ctr + 1));
    double rad = sqrt(-2.0 * log(u01(r1)));
    double ang = 6.283185307179586476925286766559 * u01(r2);
    *a = rad * cos(ang);
    *b = rad * sin(ang);
}

void syn_normal_complex(uint64_t seed, uint64_t field_id, size_t n, double *out) {
    uint64_t key = stream_key(seed, field_id);
#pragma omp parallel for schedule(static)
    for (size_t i = 0; i < n; i++) normal_pair(key, i, &out[2 * i], &out[2 * i + 1]);
}

void syn_uniform(uint64_t seed, uint64_t field_id, size_t n, double lo, double hi, double *out) {
    uint64_t key = stream_key(seed, field_id);
    for (size_t i = 0; i < n; i++) out[i] = lo + (hi - lo) * u01(mix64(key ^ mix64(i)));
}

typedef struct { double re, im; } cx;
static cx cmul(cx a, cx b) { cx r = { a.re * b.re - a.im * b.im, a.re * b.im + a.im * b.re }; return r; }
static cx cconj(cx a) { cx r = { a.re, -a.im }; return r; }

static void gram_schmidt_su3(cx *m) {
    double n0 = 0;
    for (int j = 0; j < 3; j++) n0 += m[j].re * m[j].re + m[j].im * m[j].im;
    n0 = 1.0 / sqrt(n0);
    for (int j = 0; j < 3; j++) { m[j].re *= n0; m[j].im *= n0; }
    cx d = { 0, 0 };
    for (int j = 0; j < 3; j++) { cx t = cmul(cconj(m[j]), m[3 + j]); d.re += t.re; d.im += t.im; }
    for (int j = 0; j < 3; j++) { cx t = cmul(d, m[j]); m[3 + j].re -= t.re; m[3 + j].im -= t.im; }
    double n1 = 0;
    for (int j = 0; j < 3; j++) n1 += m[3 + j].re * m[3 + j].re + m[3 + j].im * m[3 + j].im;
    n1 = 1.0 / sqrt(n1);
    for (int j = 0; j < 3; j++) { m[3 + j].re *= n1; m[3 + j].im *= n1; }
    for (int j = 0; j < 3; j++) {
        int a = (j + 1) % 3, b = (j + 2) % 3;
        cx t1 = cmul(m[a], m[3 + b]), t2 = cmul(m[b], m[3 + a]);
        cx c = { t1.re - t2.re, t1.im - t2.im };
        m[6 + j] = cconj(c);
    }
}

/* n_links Haar-like SU(3) matrices, 9 complex each */
void syn_su3_hot(uint64_t seed, uint64_t field_id, size_t n_links, double *out) {
    uint64_t key = stream_key(seed, field_id);
#pragma omp parallel for schedule(static)
    for (size_t l = 0; l < n_links; l++) {
        cx *m = (cx *)(out + l * 18);
        for (int c = 0; c < 9; c++) normal_pair(key, l * 9 + c, &m[c].re, &m[c].im);
        gram_schmidt_su3(m);
    }
}

static void mat_mul3(const cx *a, const cx *b, cx *o) {
    cx t[9];
    for (int i = 0; i < 3; i++)
        for (int j = 0; j < 3; j++) {
            cx s = { 0, 0 };
            for (int k = 0; k < 3; k++) { cx p = cmul(a[i * 3 + k], b[k * 3 + j]); s.re += p.re; s.im += p.im; }
            t[i * 3 + j] = s;
        }
    memcpy(o, t, sizeof t);
}

/* n_links matrices U = exp(i eps H), H traceless Hermitian Gaussian */
void syn_su3_warm(uint64_t seed, uint64_t field_id, size_t n_links, double eps, double *out) {
    uint64_t key = stream_key(seed, field_id);
#pragma omp parallel for schedule(static)
    for (size_t l = 0; l < n_links; l++) {
        cx A[9], X[9], T[9], E[9];
        for (int c = 0; c < 9; c++) normal_pair(key, l * 9 + c, &A[c].re, &A[c].im);
        double tr = (A[0].re + A[4].re + A[8].re) / 3.0;
        /* X = i * eps * H / 16,  H = (A + A^dag)/2 - tr/3 */
        for (int i = 0; i < 3; i++)
            for (int j = 0; j < 3; j++) {
                double hr = 0.5 * (A[i * 3 + j].re + A[j * 3 + i].re) - (i == j ? tr : 0.0);
                double hi = 0.5 * (A[i * 3 + j].im - A[j * 3 + i].im);
                X[i * 3 + j].re = -eps * hi / 16.0;
                X[i * 3 + j].im = eps * hr / 16.0;
            }
        /* Taylor series of exp(X), then square four times */
        for (int i = 0; i < 9; i++) { E[i].re = (i % 4 == 0) ? 1.0 : 0.0; E[i].im = 0.0; T[i] = E[i]; }
        for (int k = 1; k <= 18; k++) {
            mat_mul3(T, X, T);
            for (int i = 0; i < 9; i++) { T[i].re /= k; T[i].im /= k; E[i].re += T[i].re; E[i].im += T[i].im; }
        }
        for (int s = 0; s < 4; s++) mat_mul3(E, E, E);
        memcpy(out + l * 18, E, sizeof E);
    }
}
