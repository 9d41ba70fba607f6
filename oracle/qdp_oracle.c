/*
 * qdp_oracle.c -- ORACLE (test infrastructure, NOT the product).
 *
 * A plain, slow, single-threaded fp64 CPU implementation of the QDP++-style
 * lattice expressions that arXiv:1111.5596 (F. Winter, "Accelerating
 * QDP++/Chroma on GPUs") moves to the GPU: "data parallel types and
 * expressions suitable for lattice field theory" (section 1),
 * evaluated one expression at a time at every lattice site (PAPER.md:29,
 * 88-90).  The paper names the expressions only by their use ("smearing",
 * "residual calculation"); their mathematical definitions
 * are the textbook ones fixed by BASELINE.json:north_star and restated in
 * SURVEY.md section 8(c), definitions 1-6.  Each function below cites the
 * definition it writes out.
 *
 * Rules this file obeys:
 *   - Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 *     --impl reference leg may build, load or call it.
 *   - It shares no code, header, table or constant with the CUDA path under
 *     paper_1111_5596_b200/csrc/.  Neighbours are recomputed from coordinates
 *     with % at every use; there are no index tables.
 *   - No blocking, fusion or reordering: every quantity is the definition,
 *     evaluated site by site in nested loops, in the paper's host layout
 *     (site-outermost array of structures, PAPER.md:116 -- the layout the
 *     paper found un-coalesced on the device is fine for a host oracle).
 *   - Built with -O2 -ffp-contract=off: no FMA contraction, no fast-math.
 *
 * Pins (tests/test_oracle_*.py, all -m "not gpu"): unit gauge field gives
 * plaquette exactly 1 and is a fixed point of the APE step; gauge
 * invariance / covariance under random site-local SU(3); abelian closed
 * forms; plane-wave eigenvalues of hop on the unit field; hermiticity of
 * hop; scipy.linalg.polar and a Newton iteration for the projection;
 * U U^dag = 1, det U = 1 after projection; shift round trips and coordinate
 * fields; numpy brute force on 2^4 and (4,2,6,4).  Nothing here is "parity
 * unpinned".
 *
 * Host layout (the paper gives none):
 *   lex(x)   = x0 + L0*(x1 + L1*(x2 + L2*x3))        (x0 fastest)
 *   gauge    u[((lex*4 + mu)*3 + row)*3 + col]        complex = (re, im)
 *   fermion  psi[(lex*4 + spin)*3 + colour]
 *   matrix   m[(lex*3 + row)*3 + col]
 *   (U psi)_row = sum_col U[row][col] psi[col]
 * Subsets: 0 = all, 1 = even, 2 = odd; parity = (x0+x1+x2+x3) & 1
 * (SURVEY.md 8(c) reading A2).
 */
#include <math.h>
#include <stddef.h>
#include <stdint.h>
#include <string.h>

typedef struct { double re, im; } cplx;

static cplx c_add(cplx a, cplx b) { cplx r = { a.re + b.re, a.im + b.im }; return r; }
static cplx c_mul(cplx a, cplx b) {
    cplx r = { a.re * b.re - a.im * b.im, a.re * b.im + a.im * b.re };
    return r;
}
static cplx c_conj(cplx a) { cplx r = { a.re, -a.im }; return r; }
static cplx c_scale(double s, cplx a) { cplx r = { s * a.re, s * a.im }; return r; }

/* 3x3 complex matrices, row-major m[row*3+col]. */
static void m_mul(const cplx *a, const cplx *b, cplx *out) {
    cplx t[9];
    for (int i = 0; i < 3; i++)
        for (int j = 0; j < 3; j++) {
            cplx s = { 0.0, 0.0 };
            for (int k = 0; k < 3; k++) s = c_add(s, c_mul(a[i * 3 + k], b[k * 3 + j]));
            t[i * 3 + j] = s;
        }
    memcpy(out, t, sizeof t);
}
static void m_adj(const cplx *a, cplx *out) {
    cplx t[9];
    for (int i = 0; i < 3; i++)
        for (int j = 0; j < 3; j++) t[i * 3 + j] = c_conj(a[j * 3 + i]);
    memcpy(out, t, sizeof t);
}
static cplx m_trace(const cplx *a) { return c_add(c_add(a[0], a[4]), a[8]); }
static cplx m_det(const cplx *a) {
    cplx t0 = c_mul(a[0], c_add(c_mul(a[4], a[8]), c_scale(-1.0, c_mul(a[5], a[7]))));
    cplx t1 = c_mul(a[1], c_add(c_mul(a[3], a[8]), c_scale(-1.0, c_mul(a[5], a[6]))));
    cplx t2 = c_mul(a[2], c_add(c_mul(a[3], a[7]), c_scale(-1.0, c_mul(a[4], a[6]))));
    return c_add(c_add(t0, c_scale(-1.0, t1)), t2);
}

/* ---- geometry ---------------------------------------------------------- */

static size_t volume(const int *L) { return (size_t)L[0] * L[1] * L[2] * L[3]; }
static void coords_of(const int *L, size_t lex, int *x) {
    x[0] = (int)(lex % L[0]); lex /= L[0];
    x[1] = (int)(lex % L[1]); lex /= L[1];
    x[2] = (int)(lex % L[2]); lex /= L[2];
    x[3] = (int)lex;
}
static size_t lex_of(const int *L, const int *x) {
    return (size_t)x[0] + (size_t)L[0] * (x[1] + (size_t)L[1] * (x[2] + (size_t)L[2] * x[3]));
}
/* lex index of x + step*mu_hat, coordinates mod L (periodic). Definition 1. */
static size_t hop_lex(const int *L, const int *x, int mu, int step) {
    int y[4] = { x[0], x[1], x[2], x[3] };
    y[mu] = ((x[mu] + step) % L[mu] + L[mu]) % L[mu];
    return lex_of(L, y);
}
static int parity_of(const int *x) { return (x[0] + x[1] + x[2] + x[3]) & 1; }
static int in_subset(const int *x, int subset) {
    if (subset == 0) return 1;
    return parity_of(x) == (subset == 1 ? 0 : 1);
}

/* out[lex(x)] = lex(x + sign*mu_hat).  SURVEY.md Appendix A "Neighbour tables". */
void orc_neighbor_table(const int *L, int mu, int sign, int32_t *out) {
    size_t V = volume(L);
    for (size_t s = 0; s < V; s++) {
        int x[4]; coords_of(L, s, x);
        out[s] = (int32_t)hop_lex(L, x, mu, sign);
    }
}
/* mask[lex(x)] = (x0+x1+x2+x3) & 1.  Reading A2. */
void orc_parity_mask(const int *L, uint8_t *out) {
    size_t V = volume(L);
    for (size_t s = 0; s < V; s++) {
        int x[4]; coords_of(L, s, x);
        out[s] = (uint8_t)parity_of(x);
    }
}

/* ---- shift (definition 1) --------------------------------------------------
 * dst(x) = src(x + sign*mu_hat) for x in subset; other sites of dst untouched.
 * Pure data movement on opaque per-site records so it is bit-exact for any
 * element type. */
void orc_shift_bytes_range(const int *L, size_t bytes_per_site, const void *src, void *dst,
                           int mu, int sign, int subset, size_t lex_begin, size_t lex_end) {
    const char *s = (const char *)src;
    char *d = (char *)dst;
    for (size_t i = lex_begin; i < lex_end; i++) {
        int x[4]; coords_of(L, i, x);
        if (!in_subset(x, subset)) continue;
        size_t j = hop_lex(L, x, mu, sign);
        memcpy(d + i * bytes_per_site, s + j * bytes_per_site, bytes_per_site);
    }
}
void orc_shift_bytes(const int *L, size_t bytes_per_site, const void *src, void *dst,
                     int mu, int sign, int subset) {
    orc_shift_bytes_range(L, bytes_per_site, src, dst, mu, sign, subset, 0, volume(L));
}

/* ---- plaquette (definition 2) ------------------------------------------- */

static const cplx *link_at(const double *u, size_t lex, int mu) {
    return (const cplx *)(u + ((lex * 4 + (size_t)mu) * 9) * 2);
}

/* Re tr P_{mu nu}(x), P = U_mu(x) U_nu(x+mu) U_mu(x+nu)^dag U_nu(x)^dag. */
static double plaq_retr(const int *L, const double *u, const int *x, int mu, int nu) {
    size_t s = lex_of(L, x);
    cplx a[9], b[9], t[9];
    m_mul(link_at(u, s, mu), link_at(u, hop_lex(L, x, mu, +1), nu), a);
    m_adj(link_at(u, hop_lex(L, x, nu, +1), mu), b);
    m_mul(a, b, t);
    m_adj(link_at(u, s, nu), b);
    m_mul(t, b, a);
    return m_trace(a).re;
}

/* out6 = Re tr P_{mu nu}(x) for (mu,nu) = (0,1),(0,2),(1,2),(0,3),(1,3),(2,3). */
void orc_plaquette_site(const int *L, const double *u, size_t lex, double *out6) {
    static const int pl[6][2] = { {0,1}, {0,2}, {1,2}, {0,3}, {1,3}, {2,3} };
    int x[4]; coords_of(L, lex, x);
    for (int p = 0; p < 6; p++) out6[p] = plaq_retr(L, u, x, pl[p][0], pl[p][1]);
}

/* Compensated (Neumaier) accumulator: the oracle's global sums do not depend
 * on summation order to the precision the parity bar needs (reading A12). */
typedef struct { double s, c; } ksum;
static void k_add(ksum *k, double v) {
    double t = k->s + v;
    if (fabs(k->s) >= fabs(v)) k->c += (k->s - t) + v; else k->c += (v - t) + k->s;
    k->s = t;
}
static double k_val(const ksum *k) { return k->s + k->c; }

/* out[0] = (1/(6*3*N)) sum_{x in sub} sum_{mu<nu} Re tr P_{mu nu}(x)
 * out[1] = the 3 spatial planes (mu<nu<3), normalised 1/(3*3*N)
 * out[2] = the 3 temporal planes (nu=3),   normalised 1/(3*3*N)
 * N = number of sites in the subset (reading A4, A5). */
/* The same sums restricted to lex sites [lex_begin, lex_end): out3 gets the three
 * normalised values with N = subset sites in the range.  orc_plaquette is the full
 * range.  (Used by bench.py to time a bounded sample of a large lattice.) */
void orc_plaquette_range(const int *L, const double *u, int subset, size_t lex_begin,
                         size_t lex_end, double *out3) {
    size_t n = 0;
    ksum ss = { 0, 0 }, st = { 0, 0 };
    for (size_t s = lex_begin; s < lex_end; s++) {
        int x[4]; coords_of(L, s, x);
        if (!in_subset(x, subset)) continue;
        n++;
        for (int mu = 0; mu < 4; mu++)
            for (int nu = mu + 1; nu < 4; nu++) {
                double v = plaq_retr(L, u, x, mu, nu);
                if (nu == 3) k_add(&st, v); else k_add(&ss, v);
            }
    }
    double sp = k_val(&ss), tp = k_val(&st), N = (double)n;
    out3[0] = (sp + tp) / (6.0 * 3.0 * N);
    out3[1] = sp / (3.0 * 3.0 * N);
    out3[2] = tp / (3.0 * 3.0 * N);
}
void orc_plaquette(const int *L, const double *u, int subset, double *out3) {
    orc_plaquette_range(L, u, subset, 0, volume(L), out3);
}

/* ---- SU(3) projection (definition 4, Appendix B) -------------------------- */

/* Cyclic complex Jacobi on a 3x3 Hermitian H: H = Q diag(lam) Q^dag.
 * Each rotation is applied as plain J^dag H J, Q <- Q J with full 3x3 products. */
static void herm_eig3(const cplx *Hin, double *lam, cplx *Q) {
    cplx H[9];
    memcpy(H, Hin, sizeof H);
    for (int i = 0; i < 9; i++) { Q[i].re = (i % 4 == 0) ? 1.0 : 0.0; Q[i].im = 0.0; }
    double tr = H[0].re + H[4].re + H[8].re;
    for (int sweep = 0; sweep < 100; sweep++) {
        double off = 0.0;
        for (int p = 0; p < 3; p++)
            for (int q = p + 1; q < 3; q++)
                off += H[p * 3 + q].re * H[p * 3 + q].re + H[p * 3 + q].im * H[p * 3 + q].im;
        if (sqrt(off) <= 1e-17 * fabs(tr)) break;
        for (int p = 0; p < 3; p++)
            for (int q = p + 1; q < 3; q++) {
                cplx g = H[p * 3 + q];
                double ag = sqrt(g.re * g.re + g.im * g.im);
                if (ag == 0.0) continue;
                double a = H[p * 3 + p].re, b = H[q * 3 + q].re;
                /* phase e^{i phi} of g, then a real 2x2 Jacobi rotation */
                cplx eph = { g.re / ag, g.im / ag };
                double tau = (b - a) / (2.0 * ag);
                double t = (tau >= 0.0 ? 1.0 : -1.0) / (fabs(tau) + sqrt(1.0 + tau * tau));
                double c = 1.0 / sqrt(1.0 + t * t), s = t * c;
                cplx J[9], Jd[9], T[9];
                for (int i = 0; i < 9; i++) { J[i].re = (i % 4 == 0) ? 1.0 : 0.0; J[i].im = 0.0; }
                /* J = D R, D = diag(1, e^{-i phi}) on (p,q), R = [[c, s], [-s, c]] */
                J[p * 3 + p].re = c;  J[p * 3 + p].im = 0.0;
                J[p * 3 + q].re = s;  J[p * 3 + q].im = 0.0;
                J[q * 3 + p] = c_scale(-s, c_conj(eph));
                J[q * 3 + q] = c_scale(c, c_conj(eph));
                m_adj(J, Jd);
                m_mul(Jd, H, T);
                m_mul(T, J, H);
                m_mul(Q, J, Q);
                /* the rotated pair is annihilated up to rounding: set it to exactly 0
                 * (standard Jacobi practice) and keep H exactly Hermitian */
                H[p * 3 + q].re = 0.0; H[p * 3 + q].im = 0.0;
                for (int i = 0; i < 3; i++) {
                    H[i * 3 + i].im = 0.0;
                    for (int j = i + 1; j < 3; j++) H[j * 3 + i] = c_conj(H[i * 3 + j]);
                }
            }
    }
    lam[0] = H[0].re; lam[1] = H[4].re; lam[2] = H[8].re;
}

/* W = V (V^dag V)^{-1/2}: the unitary polar factor (definition 4). */
void orc_polar_unitary(const double *Vin, double *Wout) {
    const cplx *V = (const cplx *)Vin;
    cplx Vd[9], H[9], Q[9], Qd[9], D[9], R[9], T[9], W[9];
    double lam[3];
    m_adj(V, Vd);
    m_mul(Vd, V, H);
    herm_eig3(H, lam, Q);
    memset(D, 0, sizeof D);
    for (int k = 0; k < 3; k++) D[k * 4].re = 1.0 / sqrt(lam[k]);
    m_adj(Q, Qd);
    m_mul(Q, D, T);
    m_mul(T, Qd, R);
    m_mul(V, R, W);
    memcpy(Wout, W, sizeof W);
}

/* Proj(V) = W e^{-i theta/3}, theta = arg det V in (-pi, pi] (readings A8, A9). */
void orc_proj_su3(const double *Vin, double *out) {
    cplx W[9];
    orc_polar_unitary(Vin, (double *)W);
    cplx d = m_det((const cplx *)Vin);
    double theta = atan2(d.im, d.re);
    cplx ph = { cos(theta / 3.0), -sin(theta / 3.0) };
    cplx *o = (cplx *)out;
    for (int i = 0; i < 9; i++) o[i] = c_mul(W[i], ph);
}

/* ---- one binary colour-matrix expression (first step) -------------------
 *   dst(x) = opA(A(x)) * opB(B(x + sign*mu)),   op = identity (0) or adjoint (1),   x in subset;
 * mu = -1: no shift.  A, B, dst are arrays of `na`, `nb`, `nd` matrices per site of which matrix
 * `ia`, `ib`, `id` takes part (a colour-matrix field has 1, a gauge field 4: "U_mu" is matrix mu).
 * This is the building block of QDP++ expressions such as  m = u[mu] * shift(u[nu], FORWARD, mu). */
void orc_matmul(const int *L, double *dst, int nd, int id, const double *A, int na, int ia, int adj_a,
                const double *B, int nb, int ib, int adj_b, int mu, int sign, int subset) {
    for (size_t s = 0; s < volume(L); s++) {
        int x[4]; coords_of(L, s, x);
        if (!in_subset(x, subset)) continue;
        size_t sbn = mu < 0 ? s : hop_lex(L, x, mu, sign);
        const cplx *a = (const cplx *)A + (s * na + ia) * 9, *b = (const cplx *)B + (sbn * nb + ib) * 9;
        cplx ta[9], tb[9], r[9];
        if (adj_a) m_adj(a, ta); else memcpy(ta, a, sizeof ta);
        if (adj_b) m_adj(b, tb); else memcpy(tb, b, sizeof tb);
        m_mul(ta, tb, r);
        memcpy((cplx *)dst + (s * nd + id) * 9, r, sizeof r);
    }
}

/* chi(x) = opA(A(x)) psi(x + sign*mu) on the subset: colour matrix (slot ia of na per site) times
 * the colour index of every spin component of a fermion; op = identity or adjoint; mu = -1: no shift.
 * ("colour-matrix x fermion on arbitrary fields, shift of leaves".) */
void orc_matvec(const int *L, double *chi, const double *A, int na, int ia, int adj_a, const double *psi,
                int mu, int sign, int subset) {
    for (size_t s = 0; s < volume(L); s++) {
        int x[4]; coords_of(L, s, x);
        if (!in_subset(x, subset)) continue;
        size_t sn = mu < 0 ? s : hop_lex(L, x, mu, sign);
        const cplx *a = (const cplx *)A + (s * na + ia) * 9, *p = (const cplx *)psi + sn * 12;
        cplx ta[9], r[12];
        if (adj_a) m_adj(a, ta); else memcpy(ta, a, sizeof ta);
        for (int sp = 0; sp < 4; sp++)
            for (int i = 0; i < 3; i++) {
                cplx acc = { 0, 0 };
                for (int j = 0; j < 3; j++) acc = c_add(acc, c_mul(ta[i * 3 + j], p[sp * 3 + j]));
                r[sp * 3 + i] = acc;
            }
        memcpy((cplx *)chi + s * 12, r, sizeof r);
    }
}

/* ---- trace / real and the whole-field forms used by the expression layer ("adj, trace, real,
 * colour-matrix x colour-matrix on arbitrary fields, shift of leaves"; expressions that look like
 * their mathematical counterparts, evaluated site by site without temporaries) -----------------------------------
 *   orc_trace_mul:       out(x) = tr[ opA(A(x)) opB(B(x + sign*mu)) ]   one complex number per site, x in subset;
 *                        real(...) of it is the .re member (the QDP++ `real`), taken by the caller.
 *   orc_staple_field:    out(x) = S_mu(x) of orc_staple_site, a colour-matrix field, x in subset.
 *   orc_ape_blend_field: out(x) = (1-alpha) U_mu(x) + (alpha/n) S_mu(x), x in subset.
 * Sites outside the subset keep their previous contents of `out`. */
void orc_trace_mul(const int *L, double *out, const double *A, int na, int ia, int adj_a,
                   const double *B, int nb, int ib, int adj_b, int mu, int sign, int subset) {
    for (size_t s = 0; s < volume(L); s++) {
        int x[4]; coords_of(L, s, x);
        if (!in_subset(x, subset)) continue;
        size_t sbn = mu < 0 ? s : hop_lex(L, x, mu, sign);
        const cplx *a = (const cplx *)A + (s * na + ia) * 9, *b = (const cplx *)B + (sbn * nb + ib) * 9;
        cplx ta[9], tb[9], r[9];
        if (adj_a) m_adj(a, ta); else memcpy(ta, a, sizeof ta);
        if (adj_b) m_adj(b, tb); else memcpy(tb, b, sizeof tb);
        m_mul(ta, tb, r);
        ((cplx *)out)[s] = m_trace(r);
    }
}
/* ---- reunitarisation of whole fields (alternative projections) ----------
 * Gram-Schmidt: row0 = v0/|v0|; row1 = v1 - (row0 . v1) row0, normalised, with (a . b) = sum_j conj(a_j) b_j;
 * row2 = conj(row0 x row1).  The result is in SU(3) by construction; unlike Proj it is not gauge
 * covariant (reading A8), which is why the APE step does not use it. */
void orc_gram_schmidt_su3(const double *Vin, double *out) {
    const cplx *v = (const cplx *)Vin;
    cplx r[9];
    double n0 = 0;
    for (int j = 0; j < 3; j++) n0 += v[j].re * v[j].re + v[j].im * v[j].im;
    n0 = sqrt(n0);
    for (int j = 0; j < 3; j++) r[j] = c_scale(1.0 / n0, v[j]);
    cplx dot = { 0, 0 };
    for (int j = 0; j < 3; j++) dot = c_add(dot, c_mul(c_conj(r[j]), v[3 + j]));
    double n1 = 0;
    for (int j = 0; j < 3; j++) {
        cplx t = c_mul(dot, r[j]);
        r[3 + j].re = v[3 + j].re - t.re;
        r[3 + j].im = v[3 + j].im - t.im;
        n1 += r[3 + j].re * r[3 + j].re + r[3 + j].im * r[3 + j].im;
    }
    n1 = sqrt(n1);
    for (int j = 0; j < 3; j++) r[3 + j] = c_scale(1.0 / n1, r[3 + j]);
    for (int j = 0; j < 3; j++) {
        int a = (j + 1) % 3, b = (j + 2) % 3;
        cplx x = c_mul(r[a], r[3 + b]), y = c_mul(r[b], r[3 + a]);
        cplx c = { x.re - y.re, x.im - y.im };
        r[6 + j] = c_conj(c);
    }
    memcpy(out, r, sizeof r);
}

/* out(x) = method(in(x)) for every 3x3 matrix of the sites in the subset; method 0 = Proj
 * (definition 4), 1 = Gram-Schmidt.  nmat = matrices per site (4 for a gauge field, 1 for a colour
 * matrix).  Sites outside the subset keep what `out` held. */
void orc_reunitarize(const int *L, int nmat, const double *in, double *out, int method, int subset) {
    for (size_t s = 0; s < volume(L); s++) {
        int x[4]; coords_of(L, s, x);
        if (!in_subset(x, subset)) continue;
        for (int m = 0; m < nmat; m++) {
            const double *vi = in + (s * nmat + m) * 18;
            double *vo = out + (s * nmat + m) * 18;
            if (method == 0) orc_proj_su3(vi, vo); else orc_gram_schmidt_su3(vi, vo);
        }
    }
}

/* ---- iterative max-Re-tr projection ("iterative max-Re-tr"; Cabibbo-Marinari sweeps) -----
 * Finds X in SU(3) that increases Re tr(X V^dag) by exact maximisation over one SU(2) subgroup at a time.
 * Reading (f2): X_0 = Gram-Schmidt(V); one iteration = the three subgroups acting on the index
 * pairs (0,1), (1,2), (0,2) in that order.  For the pair (i,j) let M = X V^dag and m its 2x2 block
 * [[M_ii, M_ij], [M_ji, M_jj]].  Writing m = alpha_0 1 + sum_k alpha_k sigma_k with complex alpha and an SU(2) element
 * a = a_0 1 + i sum_k a_k sigma_k (a real, |a| = 1):  Re tr(a m) = 2 (a_0 Re alpha_0 - sum_k a_k Im alpha_k), which is
 * maximal for (a_0, a_k) = (Re alpha_0, -Im alpha_k) / norm, i.e. with
 *     r0 = Re(m00 + m11), r1 = -Im(m01 + m10), r2 = -Re(m01 - m10), r3 = -Im(m00 - m11)
 *     a = [[r0 + i r3, r2 + i r1], [-r2 + i r1, r0 - i r3]] / |r|.
 * X <- A X, A = a embedded in rows/columns (i,j).  Every update leaves X in SU(3) and cannot decrease Re tr(X V^dag).
 * retr (nullable) receives Re tr(X V^dag) after X_0 and after each of the 3*iters updates (1 + 3*iters values). */
void orc_max_retr_su3(const double *Vin, int iters, double *out, double *retr) {
    const cplx *V = (const cplx *)Vin;
    cplx X[9], Vd[9], M[9];
    orc_gram_schmidt_su3(Vin, (double *)X);
    m_adj(V, Vd);
    int nrec = 0;
    m_mul(X, Vd, M);
    if (retr) retr[nrec++] = m_trace(M).re;
    static const int pi[3] = { 0, 1, 0 }, pj[3] = { 1, 2, 2 };
    for (int it = 0; it < iters; it++)
        for (int sg = 0; sg < 3; sg++) {
            const int i = pi[sg], j = pj[sg];
            m_mul(X, Vd, M);
            const cplx m00 = M[i * 3 + i], m01 = M[i * 3 + j], m10 = M[j * 3 + i], m11 = M[j * 3 + j];
            double r0 = m00.re + m11.re, r1 = -(m01.im + m10.im), r2 = -(m01.re - m10.re), r3 = -(m00.im - m11.im);
            const double nr = sqrt(r0 * r0 + r1 * r1 + r2 * r2 + r3 * r3);
            if (nr > 0) { r0 /= nr; r1 /= nr; r2 /= nr; r3 /= nr; } else { r0 = 1; r1 = r2 = r3 = 0; }
            const cplx a00 = { r0, r3 }, a01 = { r2, r1 }, a10 = { -r2, r1 }, a11 = { r0, -r3 };
            for (int c = 0; c < 3; c++) {          /* rows i and j of X are mixed */
                const cplx xi = X[i * 3 + c], xj = X[j * 3 + c];
                X[i * 3 + c] = c_add(c_mul(a00, xi), c_mul(a01, xj));
                X[j * 3 + c] = c_add(c_mul(a10, xi), c_mul(a11, xj));
            }
            if (retr) { m_mul(X, Vd, M); retr[nrec++] = m_trace(M).re; }
        }
    memcpy(out, X, sizeof X);
}
/* whole fields: out(x) = orc_max_retr_su3(in(x)) for every matrix of the subset's sites (nmat per site) */
void orc_project_max_retr(const int *L, int nmat, const double *in, double *out, int iters, int subset) {
    for (size_t s = 0; s < volume(L); s++) {
        int x[4]; coords_of(L, s, x);
        if (!in_subset(x, subset)) continue;
        for (int m = 0; m < nmat; m++)
            orc_max_retr_su3(in + (s * nmat + m) * 18, iters, out + (s * nmat + m) * 18, NULL);
    }
}

/* smallest singular value^2 of V (lambda_min of V^dag V), for reading A10 */
double orc_min_eig_vdv(const double *Vin) {
    const cplx *V = (const cplx *)Vin;
    cplx Vd[9], H[9], Q[9];
    double lam[3];
    m_adj(V, Vd);
    m_mul(Vd, V, H);
    herm_eig3(H, lam, Q);
    double m = lam[0];
    if (lam[1] < m) m = lam[1];
    if (lam[2] < m) m = lam[2];
    return m;
}

/* ---- staples and the APE step (definition 3) ------------------------------ */

/* S_mu(x) = sum_{nu in smeared set, nu != mu}
 *   [ U_nu(x) U_mu(x+nu) U_nu(x+mu)^dag + U_nu(x-nu)^dag U_mu(x-nu) U_nu(x-nu+mu) ]
 * smeared set = {0,1,2} if t_dir == 3, {0,1,2,3} if t_dir == -1.
 * Returns the number of staples n = 2*(|set|-1). */
int orc_staple_site(const int *L, const double *u, size_t lex, int mu, int t_dir, double *S18) {
    int x[4]; coords_of(L, lex, x);
    cplx S[9];
    memset(S, 0, sizeof S);
    int n = 0;
    for (int nu = 0; nu < 4; nu++) {
        if (nu == mu || nu == t_dir) continue;
        cplx a[9], b[9], t[9];
        /* upper: U_nu(x) U_mu(x+nu) U_nu(x+mu)^dag */
        m_mul(link_at(u, lex, nu), link_at(u, hop_lex(L, x, nu, +1), mu), a);
        m_adj(link_at(u, hop_lex(L, x, mu, +1), nu), b);
        m_mul(a, b, t);
        for (int i = 0; i < 9; i++) S[i] = c_add(S[i], t[i]);
        /* lower: U_nu(x-nu)^dag U_mu(x-nu) U_nu(x-nu+mu) */
        int y[4] = { x[0], x[1], x[2], x[3] };
        y[nu] = ((x[nu] - 1) % L[nu] + L[nu]) % L[nu];
        size_t ly = lex_of(L, y);
        m_adj(link_at(u, ly, nu), b);
        m_mul(b, link_at(u, ly, mu), a);
        m_mul(a, link_at(u, hop_lex(L, y, mu, +1), nu), t);
        for (int i = 0; i < 9; i++) S[i] = c_add(S[i], t[i]);
        n += 2;
    }
    memcpy(S18, S, sizeof S);
    return n;
}

/* V_mu(x) = (1-alpha) U_mu(x) + (alpha/n) S_mu(x)  (reading A6), before projection. */
void orc_ape_blend_site(const int *L, const double *u, size_t lex, int mu, double alpha,
                        int t_dir, double *V18) {
    cplx S[9];
    int n = orc_staple_site(L, u, lex, mu, t_dir, (double *)S);
    const cplx *U = link_at(u, lex, mu);
    cplx *V = (cplx *)V18;
    for (int i = 0; i < 9; i++)
        V[i] = c_add(c_scale(1.0 - alpha, U[i]), c_scale(alpha / (double)n, S[i]));
}

/* U'_mu(x) = Proj(V_mu(x)); if mu == t_dir the link is copied unchanged (A7). */
void orc_ape_site(const int *L, const double *u, size_t lex, int mu, double alpha, int t_dir,
                  double *out18) {
    if (mu == t_dir) { memcpy(out18, link_at(u, lex, mu), 18 * sizeof(double)); return; }
    double V[18];
    orc_ape_blend_site(L, u, lex, mu, alpha, t_dir, V);
    orc_proj_su3(V, out18);
}

/* whole-field forms of the two functions above (expression layer, row f1; see orc_trace_mul) */
void orc_staple_field(const int *L, const double *u, int mu, int t_dir, int subset, double *out) {
    for (size_t s = 0; s < volume(L); s++) {
        int x[4]; coords_of(L, s, x);
        if (!in_subset(x, subset)) continue;
        orc_staple_site(L, u, s, mu, t_dir, out + s * 18);
    }
}
void orc_ape_blend_field(const int *L, const double *u, int mu, double alpha, int t_dir, int subset, double *out) {
    for (size_t s = 0; s < volume(L); s++) {
        int x[4]; coords_of(L, s, x);
        if (!in_subset(x, subset)) continue;
        orc_ape_blend_site(L, u, s, mu, alpha, t_dir, out + s * 18);
    }
}

void orc_ape_smear_step_range(const int *L, const double *u_in, double *u_out, double alpha,
                              int t_dir, int subset, size_t lex_begin, size_t lex_end) {
    for (size_t s = lex_begin; s < lex_end; s++) {
        int x[4]; coords_of(L, s, x);
        if (!in_subset(x, subset)) continue;
        for (int mu = 0; mu < 4; mu++)
            orc_ape_site(L, u_in, s, mu, alpha, t_dir, u_out + ((s * 4 + (size_t)mu) * 9) * 2);
    }
}
void orc_ape_smear_step(const int *L, const double *u_in, double *u_out, double alpha, int t_dir,
                        int subset) {
    orc_ape_smear_step_range(L, u_in, u_out, alpha, t_dir, subset, 0, volume(L));
}

/* ---- hop (definition 5) ---------------------------------------------------
 * chi(x)_{s a} = sum_mu sum_b [ U_mu(x)_{ab} psi(x+mu)_{sb}
 *                             + conj(U_mu(x-mu)_{ba}) psi(x-mu)_{sb} ]      */
/* hop restricted to the directions mu != t_dir (t_dir = -1: all four) */
void orc_hop_site_dirs(const int *L, const double *u, const double *psi, size_t lex, int t_dir,
                       double *out24) {
    int x[4]; coords_of(L, lex, x);
    cplx chi[12];
    memset(chi, 0, sizeof chi);
    for (int mu = 0; mu < 4; mu++) {
        if (mu == t_dir) continue;
        size_t lf = hop_lex(L, x, mu, +1), lb = hop_lex(L, x, mu, -1);
        const cplx *Uf = link_at(u, lex, mu), *Ub = link_at(u, lb, mu);
        const cplx *pf = (const cplx *)(psi + lf * 24), *pb = (const cplx *)(psi + lb * 24);
        for (int s = 0; s < 4; s++)
            for (int a = 0; a < 3; a++)
                for (int b = 0; b < 3; b++) {
                    chi[s * 3 + a] = c_add(chi[s * 3 + a], c_mul(Uf[a * 3 + b], pf[s * 3 + b]));
                    chi[s * 3 + a] = c_add(chi[s * 3 + a], c_mul(c_conj(Ub[b * 3 + a]), pb[s * 3 + b]));
                }
    }
    memcpy(out24, chi, sizeof chi);
}
void orc_hop_site(const int *L, const double *u, const double *psi, size_t lex, double *out24) {
    orc_hop_site_dirs(L, u, psi, lex, -1, out24);
}

void orc_hop_range(const int *L, const double *u, const double *psi, double *chi, int subset,
                   size_t lex_begin, size_t lex_end) {
    for (size_t s = lex_begin; s < lex_end; s++) {
        int x[4]; coords_of(L, s, x);
        if (!in_subset(x, subset)) continue;
        orc_hop_site(L, u, psi, s, chi + s * 24);
    }
}
void orc_hop(const int *L, const double *u, const double *psi, double *chi, int subset) {
    orc_hop_range(L, u, psi, chi, subset, 0, volume(L));
}

/* chi = a psi + b hop(psi) on the subset (definition 6, axpy_hop). */
void orc_axpy_hop_range(const int *L, double a, double b, const double *u, const double *psi,
                        double *chi, int subset, size_t lex_begin, size_t lex_end) {
    for (size_t s = lex_begin; s < lex_end; s++) {
        int x[4]; coords_of(L, s, x);
        if (!in_subset(x, subset)) continue;
        double h[24];
        orc_hop_site(L, u, psi, s, h);
        for (int i = 0; i < 24; i++) chi[s * 24 + i] = a * psi[s * 24 + i] + b * h[i];
    }
}
void orc_axpy_hop(const int *L, double a, double b, const double *u, const double *psi,
                  double *chi, int subset) {
    orc_axpy_hop_range(L, a, b, u, psi, chi, subset, 0, volume(L));
}

/* ---- quark smearing step (the SRC/SNK smearing stage of PAPER.md:82, 106) --
 * chi(x) = a psi(x) + b sum_{mu != t_dir} [ U_mu(x) psi(x+mu) + U_mu(x-mu)^dag psi(x-mu) ]
 * on the subset: one step of gauge-covariant Wuppertal / Gaussian smearing for t_dir = 3
 * (spatial hops only); t_dir = -1 is definition 6 (axpy_hop). */
void orc_smear_hop_range(const int *L, double a, double b, const double *u, const double *psi,
                         double *chi, int t_dir, int subset, size_t lex_begin, size_t lex_end) {
    for (size_t s = lex_begin; s < lex_end; s++) {
        int x[4]; coords_of(L, s, x);
        if (!in_subset(x, subset)) continue;
        double h[24];
        orc_hop_site_dirs(L, u, psi, s, t_dir, h);
        for (int i = 0; i < 24; i++) chi[s * 24 + i] = a * psi[s * 24 + i] + b * h[i];
    }
}
void orc_smear_hop(const int *L, double a, double b, const double *u, const double *psi,
                   double *chi, int t_dir, int subset) {
    orc_smear_hop_range(L, a, b, u, psi, chi, t_dir, subset, 0, volume(L));
}

/* ---- global reductions (definition 6) -------------------------------------
 * reals = 2 * (complex components per site). Lexicographic order, compensated. */
double orc_norm2_range(const int *L, int reals, const double *f, int subset, size_t lex_begin,
                       size_t lex_end) {
    ksum k = { 0, 0 };
    for (size_t s = lex_begin; s < lex_end; s++) {
        int x[4]; coords_of(L, s, x);
        if (!in_subset(x, subset)) continue;
        for (int i = 0; i < reals; i++) k_add(&k, f[s * reals + i] * f[s * reals + i]);
    }
    return k_val(&k);
}
double orc_norm2(const int *L, int reals, const double *f, int subset) {
    return orc_norm2_range(L, reals, f, subset, 0, volume(L));
}

/* out = sum_x sum_c conj(a_c(x)) b_c(x)  (conjugates its FIRST argument, A12). */
void orc_inner_range(const int *L, int reals, const double *a, const double *b, int subset,
                     size_t lex_begin, size_t lex_end, double *out2) {
    ksum kr = { 0, 0 }, ki = { 0, 0 };
    for (size_t s = lex_begin; s < lex_end; s++) {
        int x[4]; coords_of(L, s, x);
        if (!in_subset(x, subset)) continue;
        for (int c = 0; c < reals / 2; c++) {
            cplx p = c_mul(c_conj(((const cplx *)a)[s * (reals / 2) + c]),
                           ((const cplx *)b)[s * (reals / 2) + c]);
            k_add(&kr, p.re);
            k_add(&ki, p.im);
        }
    }
    out2[0] = k_val(&kr);
    out2[1] = k_val(&ki);
}
void orc_inner(const int *L, int reals, const double *a, const double *b, int subset, double *out2) {
    orc_inner_range(L, reals, a, b, subset, 0, volume(L), out2);
}

/* dst = a x + b y on the subset, real a, b, any field kind (reals = 2 * complex components per
 * site): the "residual calculation and solution reconstruction" expressions of PAPER.md:96
 * (r = b - A x, x += alpha p ...).  Two roundings per term, like a*psi + b*hop in definition 6. */
void orc_axpby(const int *L, int reals, double a, const double *x, double b, const double *y,
               double *dst, int subset) {
    for (size_t s = 0; s < volume(L); s++) {
        int c[4]; coords_of(L, s, c);
        if (!in_subset(c, subset)) continue;
        for (int i = 0; i < reals; i++) dst[s * reals + i] = a * x[s * reals + i] + b * y[s * reals + i];
    }
}

/* time-slice sums, the reduction under every hadron two-point function
 * (HAD stage):
 *   out[t] = sum_{x in subset, x3 = t} sum_c conj(a_c(x)) b_c(x),   t = 0 .. L3-1   (re, im pairs).
 * With a = b a quark propagator column this is the pion correlator of that column. */
void orc_inner_timeslices(const int *L, int reals, const double *a, const double *b, int subset,
                          double *out) {
    for (int t = 0; t < L[3]; t++) {
        ksum kr = { 0, 0 }, ki = { 0, 0 };
        for (size_t s = 0; s < volume(L); s++) {
            int x[4]; coords_of(L, s, x);
            if (x[3] != t || !in_subset(x, subset)) continue;
            for (int c = 0; c < reals / 2; c++) {
                cplx p = c_mul(c_conj(((const cplx *)a)[s * (reals / 2) + c]),
                               ((const cplx *)b)[s * (reals / 2) + c]);
                k_add(&kr, p.re);
                k_add(&ki, p.im);
            }
        }
        out[2 * t] = k_val(&kr);
        out[2 * t + 1] = k_val(&ki);
    }
}

/* ---- spin matrices (meson contractions) -----------------------------------
 * Euclidean gamma matrices in the DeGrand-Rossi basis (the convention of QDP++/Chroma):
 *   g0 = [[0,0,0,i],[0,0,i,0],[0,-i,0,0],[-i,0,0,0]]    g1 = [[0,0,0,-1],[0,0,1,0],[0,1,0,0],[-1,0,0,0]]
 *   g2 = [[0,0,i,0],[0,0,0,-i],[-i,0,0,0],[0,i,0,0]]    g3 = [[0,0,1,0],[0,0,0,1],[1,0,0,0],[0,1,0,0]]
 * Gamma(n) = g0^n0 g1^n1 g2^n2 g3^n3 with n = n0 + 2 n1 + 4 n2 + 8 n3 (Gamma(15) = gamma_5). */
static void gamma_base(int mu, cplx g[16]) {
    static const int pos[4][4] = { {3, 2, 1, 0}, {3, 2, 1, 0}, {2, 3, 0, 1}, {2, 3, 0, 1} };
    static const double re[4][4] = { {0, 0, 0, 0}, {-1, 1, 1, -1}, {0, 0, 0, 0}, {1, 1, 1, 1} };
    static const double im[4][4] = { {1, 1, -1, -1}, {0, 0, 0, 0}, {1, -1, -1, 1}, {0, 0, 0, 0} };
    memset(g, 0, 16 * sizeof(cplx));
    for (int r = 0; r < 4; r++) { g[r * 4 + pos[mu][r]].re = re[mu][r]; g[r * 4 + pos[mu][r]].im = im[mu][r]; }
}
void orc_gamma_matrix(int n, double *out32) {
    cplx acc[16], tmp[16], g[16];
    memset(acc, 0, sizeof acc);
    for (int i = 0; i < 4; i++) acc[i * 5].re = 1.0;
    for (int mu = 0; mu < 4; mu++) {
        if (!((n >> mu) & 1)) continue;
        gamma_base(mu, g);
        for (int i = 0; i < 4; i++)
            for (int j = 0; j < 4; j++) {
                cplx t = { 0, 0 };
                for (int k = 0; k < 4; k++) t = c_add(t, c_mul(acc[i * 4 + k], g[k * 4 + j]));
                tmp[i * 4 + j] = t;
            }
        memcpy(acc, tmp, sizeof acc);
    }
    memcpy(out32, acc, sizeof acc);
}
/* out[t] = sum_{x in subset, x3 = t} sum_{s' s c} conj(a_{s' c}(x)) Gamma(n)_{s' s} b_{s c}(x):
 * with a, b columns of a quark propagator, the building block of meson two-point functions. */
void orc_inner_timeslices_gamma(const int *L, const double *a, const double *b, int n, int subset,
                                double *out) {
    cplx G[16];
    orc_gamma_matrix(n, (double *)G);
    for (int t = 0; t < L[3]; t++) {
        ksum kr = { 0, 0 }, ki = { 0, 0 };
        for (size_t s = 0; s < volume(L); s++) {
            int x[4]; coords_of(L, s, x);
            if (x[3] != t || !in_subset(x, subset)) continue;
            const cplx *pa = (const cplx *)a + s * 12, *pb = (const cplx *)b + s * 12;
            for (int sp = 0; sp < 4; sp++)
                for (int c = 0; c < 3; c++) {
                    cplx gb = { 0, 0 };
                    for (int s2 = 0; s2 < 4; s2++) gb = c_add(gb, c_mul(G[sp * 4 + s2], pb[s2 * 3 + c]));
                    cplx p = c_mul(c_conj(pa[sp * 3 + c]), gb);
                    k_add(&kr, p.re);
                    k_add(&ki, p.im);
                }
        }
        out[2 * t] = k_val(&kr);
        out[2 * t + 1] = k_val(&ki);
    }
}

/* ---- baryon building block ("meson/baryon colour-spin contractions"; HAD stage) ---
 * Three quark fields contracted to a colour singlet with the antisymmetric tensor, a diquark spin matrix Gamma(n)
 * between the first two, summed over each time-slice:
 *   out[t][g] = sum_{x in subset, x3 = t} sum_{(a',b',c')} eps_{a'b'c'} sum_{a b c} eps_{abc}
 *               [ sum_{al be} q1[a']_{al a}(x) Gamma(n)_{al be} q2[b']_{be b}(x) ] q3[c']_{g c}(x),     g = 0..3 (open spin).
 * nsrc = 3: q1, q2, q3 are arrays of three fermion fields each, one per SOURCE colour (columns of a quark propagator
 * with fixed source spin), and (a',b',c') runs over the six permutations with their signs: the eps_{abc} eps_{a'b'c'}
 * colour contraction of the nucleon two-point function.  nsrc = 1: one field per quark, no source contraction (the
 * colour-singlet operator eps_{abc} (q1^T Gamma q2)_{ab} q3_c of three spinor fields).  No conjugation anywhere.
 * out: [L3][4] complex. */
void orc_baryon_timeslices(const int *L, int nsrc, const double *const *q1, const double *const *q2,
                           const double *const *q3, int n, int subset, double *out) {
    cplx G[16];
    orc_gamma_matrix(n, (double *)G);
    static const int perm[6][3] = { {0,1,2}, {1,2,0}, {2,0,1}, {0,2,1}, {2,1,0}, {1,0,2} };
    static const double psign[6] = { 1, 1, 1, -1, -1, -1 };
    const int nperm = nsrc == 3 ? 6 : 1;
    for (int t = 0; t < L[3]; t++) {
        ksum k[8];
        memset(k, 0, sizeof k);
        for (size_t s = 0; s < volume(L); s++) {
            int x[4]; coords_of(L, s, x);
            if (x[3] != t || !in_subset(x, subset)) continue;
            for (int ps = 0; ps < nperm; ps++) {
                const int sa = nsrc == 3 ? perm[ps][0] : 0, sb = nsrc == 3 ? perm[ps][1] : 0, sc = nsrc == 3 ? perm[ps][2] : 0;
                const cplx *A = (const cplx *)q1[sa] + s * 12, *B = (const cplx *)q2[sb] + s * 12,
                           *C = (const cplx *)q3[sc] + s * 12;
                for (int pc = 0; pc < 6; pc++) {                /* sink colours (a,b,c) = a permutation of (0,1,2) */
                    const int a = perm[pc][0], b = perm[pc][1], c = perm[pc][2];
                    cplx dq = { 0, 0 };                         /* q1^T Gamma q2 for colours (a, b) */
                    for (int al = 0; al < 4; al++)
                        for (int be = 0; be < 4; be++)
                            dq = c_add(dq, c_mul(c_mul(A[al * 3 + a], G[al * 4 + be]), B[be * 3 + b]));
                    for (int g = 0; g < 4; g++) {
                        cplx v = c_scale(psign[ps] * psign[pc], c_mul(dq, C[g * 3 + c]));
                        k_add(&k[2 * g], v.re);
                        k_add(&k[2 * g + 1], v.im);
                    }
                }
            }
        }
        for (int i = 0; i < 8; i++) out[t * 8 + i] = k_val(&k[i]);
    }
}

/* out[c] = sum_x f_c(x), per real component (re, im interleaved like f). */
void orc_sum(const int *L, int reals, const double *f, int subset, double *out) {
    size_t V = volume(L);
    for (int i = 0; i < reals; i++) {
        ksum k = { 0, 0 };
        for (size_t s = 0; s < V; s++) {
            int x[4]; coords_of(L, s, x);
            if (!in_subset(x, subset)) continue;
            k_add(&k, f[s * reals + i]);
        }
        out[i] = k_val(&k);
    }
}
