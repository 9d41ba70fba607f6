// su3.cuh -- per-site colour algebra in registers: 3x3 complex matrices, colour
// vectors, field loads/stores in the site-fastest SoA layout, and the SU(3)
// projection.  (8(c) definitions 2-5.)
//
// Device field layout (geom.cuh): blocked site-fastest structure of arrays,
// element(c, s) = ((s >> 5) * ncomp + c) * 32 + (s & 31), s the internal site index, complex =
// (re, im) adjacent: fp64 -> one double2 = one 128-bit access per thread, a warp moves 512
// contiguous bytes per component; fp32 -> float2, 256 contiguous bytes per warp.
#pragma once
#ifndef __CUDACC_RTC__
#include <cstdio>
#include <cuda_runtime.h>
#endif
#include "geom.cuh"

namespace qdp {

template <class T> struct Vec2;
template <> struct Vec2<float> { using type = float2; };
template <> struct Vec2<double> { using type = double2; };

template <class T> struct Cx {
    T re, im;
};

template <class T> __device__ __forceinline__ Cx<T> cx(T re, T im) { Cx<T> r; r.re = re; r.im = im; return r; }
template <class T> __device__ __forceinline__ Cx<T> operator+(Cx<T> a, Cx<T> b) { return cx<T>(a.re + b.re, a.im + b.im); }
template <class T> __device__ __forceinline__ Cx<T> operator-(Cx<T> a, Cx<T> b) { return cx<T>(a.re - b.re, a.im - b.im); }
template <class T> __device__ __forceinline__ Cx<T> operator*(Cx<T> a, Cx<T> b) {
    return cx<T>(a.re * b.re - a.im * b.im, a.re * b.im + a.im * b.re);
}
template <class T> __device__ __forceinline__ Cx<T> conj(Cx<T> a) { return cx<T>(a.re, -a.im); }
// acc += a * b
template <class T> __device__ __forceinline__ void cmad(Cx<T>& acc, Cx<T> a, Cx<T> b) {
    acc.re = fma(a.re, b.re, acc.re); acc.re = fma(-a.im, b.im, acc.re);
    acc.im = fma(a.re, b.im, acc.im); acc.im = fma(a.im, b.re, acc.im);
}
// acc += conj(a) * b
template <class T> __device__ __forceinline__ void cmad_conj_a(Cx<T>& acc, Cx<T> a, Cx<T> b) {
    acc.re = fma(a.re, b.re, acc.re); acc.re = fma(a.im, b.im, acc.re);
    acc.im = fma(a.re, b.im, acc.im); acc.im = fma(-a.im, b.re, acc.im);
}
// acc += a * conj(b)
template <class T> __device__ __forceinline__ void cmad_conj_b(Cx<T>& acc, Cx<T> a, Cx<T> b) {
    acc.re = fma(a.re, b.re, acc.re); acc.re = fma(a.im, b.im, acc.re);
    acc.im = fma(a.im, b.re, acc.im); acc.im = fma(-a.re, b.im, acc.im);
}

template <class T> struct Mat3 {
    Cx<T> e[9];  // row-major e[row*3+col]
};
template <class T> struct Spinor {
    Cx<T> e[12];  // e[spin*3+colour]
};

// ---- field access ----------------------------------------------------------
// Blocked layout (geom.cuh): element(c, s) = ((s >> 5) * ncomp + c) * 32 + (s & 31).
// site_ptr() is the one address computation per (site, first component); the other
// components are at compile-time offsets of 32 elements (512 B fp64, 256 B fp32).
constexpr int kLane = 32;   // sites per block

template <class T2>
__device__ __forceinline__ T2* site_ptr_raw(T2* f, int ncomp, int c0, int s) {
    return f + ((size_t)(s >> 5) * ncomp + c0) * kLane + (s & 31);
}
#ifdef QDP_BOUNDS_CHECK
// Bounds-checked build (python -m paper_1111_5596_b200.build --bounds-check -> libqdp_b200_bc.so; compute-sanitizer is
// closed on this GPU pool): every site address is validated against the lattice in scope (`g`): the site index
// must be a real site of one of the two parity halves (not a padding lane) and the first component must lie inside
// the site.  A violation is reported through device printf ("QDP_BOUNDS ...") and the access is redirected to site 0,
// so the run continues without an illegal access and tests/test_gpu_bounds.py can count the reports.
template <class T2>
__device__ __noinline__ T2* site_ptr_checked(const Geom& g, T2* f, int ncomp, int c0, int s, int line) {
    const int hs = s >= g.Vhp ? s - g.Vhp : s;
    if (s < 0 || s >= 2 * g.Vhp || hs >= g.Vh || c0 < 0 || c0 >= ncomp) {
        printf("QDP_BOUNDS line %d: site %d (Vhp %d, Vh %d) component %d of %d\n", line, s, g.Vhp, g.Vh, c0, ncomp);
        s = 0; c0 = 0;
    }
    return site_ptr_raw(f, ncomp, c0, s);
}
#define site_ptr(f, ncomp, c0, s) ::qdp::site_ptr_checked(g, (f), (ncomp), (c0), (s), __LINE__)
#else
#define site_ptr(f, ncomp, c0, s) ::qdp::site_ptr_raw((f), (ncomp), (c0), (s))
#endif
// 3x3 matrix whose first component is at p
template <class T>
__device__ __forceinline__ Mat3<T> ld_mat_at(const typename Vec2<T>::type* __restrict__ p) {
    Mat3<T> r;
#pragma unroll
    for (int c = 0; c < 9; c++) {
        typename Vec2<T>::type v = __ldg(p + c * kLane);
        r.e[c] = cx<T>(v.x, v.y);
    }
    return r;
}
template <class T>
__device__ __forceinline__ void st_mat_at(typename Vec2<T>::type* __restrict__ p, const Mat3<T>& a) {
#pragma unroll
    for (int c = 0; c < 9; c++) {
        typename Vec2<T>::type o;
        o.x = a.e[c].re; o.y = a.e[c].im;
        p[c * kLane] = o;
    }
}
// spinor whose first component is at p
template <class T>
__device__ __forceinline__ Spinor<T> ld_spinor_at(const typename Vec2<T>::type* __restrict__ p) {
    Spinor<T> r;
#pragma unroll
    for (int c = 0; c < 12; c++) {
        typename Vec2<T>::type v = __ldg(p + c * kLane);
        r.e[c] = cx<T>(v.x, v.y);
    }
    return r;
}

// ---- matrix algebra --------------------------------------------------------
template <class T> __device__ __forceinline__ Mat3<T> mat_zero() {
    Mat3<T> r;
#pragma unroll
    for (int i = 0; i < 9; i++) r.e[i] = cx<T>(0, 0);
    return r;
}
// A * B
template <class T> __device__ __forceinline__ Mat3<T> mul(const Mat3<T>& a, const Mat3<T>& b) {
    Mat3<T> r;
#pragma unroll
    for (int i = 0; i < 3; i++)
#pragma unroll
        for (int j = 0; j < 3; j++) {
            Cx<T> s = a.e[i * 3] * b.e[j];
            cmad(s, a.e[i * 3 + 1], b.e[3 + j]);
            cmad(s, a.e[i * 3 + 2], b.e[6 + j]);
            r.e[i * 3 + j] = s;
        }
    return r;
}
// acc += A * B^dag
template <class T> __device__ __forceinline__ void mad_mul_adj(Mat3<T>& acc, const Mat3<T>& a, const Mat3<T>& b) {
#pragma unroll
    for (int i = 0; i < 3; i++)
#pragma unroll
        for (int j = 0; j < 3; j++)
#pragma unroll
            for (int k = 0; k < 3; k++) cmad_conj_b(acc.e[i * 3 + j], a.e[i * 3 + k], b.e[j * 3 + k]);
}
// A^dag * B
template <class T> __device__ __forceinline__ Mat3<T> adj_mul(const Mat3<T>& a, const Mat3<T>& b) {
    Mat3<T> r = mat_zero<T>();
#pragma unroll
    for (int i = 0; i < 3; i++)
#pragma unroll
        for (int j = 0; j < 3; j++)
#pragma unroll
            for (int k = 0; k < 3; k++) cmad_conj_a(r.e[i * 3 + j], a.e[k * 3 + i], b.e[k * 3 + j]);
    return r;
}
// acc += A * B
template <class T> __device__ __forceinline__ void mad_mul(Mat3<T>& acc, const Mat3<T>& a, const Mat3<T>& b) {
#pragma unroll
    for (int i = 0; i < 3; i++)
#pragma unroll
        for (int j = 0; j < 3; j++)
#pragma unroll
            for (int k = 0; k < 3; k++) cmad(acc.e[i * 3 + j], a.e[i * 3 + k], b.e[k * 3 + j]);
}
// ---- fp32: complex arithmetic on (re, im) register pairs with the packed instructions of sm_100 --------------------
// FFMA2 / FMUL2 work on two fp32 lanes held in an aligned register pair, and an operand may be one 32-bit register
// broadcast to both lanes or a pair with its halves swapped (SASS `R.F32`, `R.F32x2.LO_HI`).  A complex number as the
// fields store it, (re, im), is such a pair, so sum_k x_k * y_k needs no data movement at all:
//     p += x_k.re * (y_k.re, y_k.im)      q += x_k.im * (y_k.re, y_k.im)           two FFMA2 per term
//     sum x y       = (p.re - q.im, p.im + q.re) = p + (-1, +1) * swap(q)           one FFMA2
//     sum conj(x) y = (p.re + q.im, p.im - q.re) = p + (+1, -1) * swap(q)
// i.e. 7 instructions per entry of a 3x3 product where the scalar form needs 12 (2 FMUL + 10 FFMA).  Measured on
// 32^3 x 64 fp32 (profiles/r2_experiments.md): the packed instructions do not shorten the fp32 pipe time (plaquette
// 0.188 -> 0.217 ms, spatial APE 0.478 -> 0.515 ms, hop unchanged), so those kernels keep the scalar forms; the 4-D
// APE step (48 products per site, direction loop rolled) gains 11 % (0.85 -> 0.76 ms) and uses the *_pk forms below.
// Values differ from the scalar chain only in rounding order.
struct PQ { float2 p, q; };
__device__ __forceinline__ float2 f2(const Cx<float>& a) { return make_float2(a.re, a.im); }
__device__ __forceinline__ Cx<float> cxf(float2 v) { return cx<float>(v.x, v.y); }
// first term with p given (accumulate into an existing sum) or not
__device__ __forceinline__ PQ pq_first(const Cx<float>& x, const Cx<float>& y) {
    PQ s;
    s.p = __fmul2_rn(make_float2(x.re, x.re), f2(y));
    s.q = __fmul2_rn(make_float2(x.im, x.im), f2(y));
    return s;
}
__device__ __forceinline__ PQ pq_first(const Cx<float>& acc, const Cx<float>& x, const Cx<float>& y) {
    PQ s;
    s.p = __ffma2_rn(make_float2(x.re, x.re), f2(y), f2(acc));
    s.q = __fmul2_rn(make_float2(x.im, x.im), f2(y));
    return s;
}
__device__ __forceinline__ void pq_mad(PQ& s, const Cx<float>& x, const Cx<float>& y) {
    s.p = __ffma2_rn(make_float2(x.re, x.re), f2(y), s.p);
    s.q = __ffma2_rn(make_float2(x.im, x.im), f2(y), s.q);
}
__device__ __forceinline__ Cx<float> pq_sum(const PQ& s) {        // sum x y
    return cxf(__ffma2_rn(make_float2(s.q.y, s.q.x), make_float2(-1.0f, 1.0f), s.p));
}
__device__ __forceinline__ Cx<float> pq_sum_conj(const PQ& s) {   // sum conj(x) y
    return cxf(__ffma2_rn(make_float2(s.q.y, s.q.x), make_float2(1.0f, -1.0f), s.p));
}
// A * B
__device__ __forceinline__ Mat3<float> mul_pk(const Mat3<float>& a, const Mat3<float>& b) {
    Mat3<float> r;
#pragma unroll
    for (int i = 0; i < 3; i++)
#pragma unroll
        for (int j = 0; j < 3; j++) {
            PQ s = pq_first(a.e[i * 3], b.e[j]);
            pq_mad(s, a.e[i * 3 + 1], b.e[3 + j]);
            pq_mad(s, a.e[i * 3 + 2], b.e[6 + j]);
            r.e[i * 3 + j] = pq_sum(s);
        }
    return r;
}
// acc += A * B^dag:  sum_k a_ik conj(b_jk) = sum_k conj(b_jk) a_ik
__device__ __forceinline__ void mad_mul_adj_pk(Mat3<float>& acc, const Mat3<float>& a, const Mat3<float>& b) {
#pragma unroll
    for (int i = 0; i < 3; i++)
#pragma unroll
        for (int j = 0; j < 3; j++) {
            PQ s = pq_first(acc.e[i * 3 + j], b.e[j * 3], a.e[i * 3]);
            pq_mad(s, b.e[j * 3 + 1], a.e[i * 3 + 1]);
            pq_mad(s, b.e[j * 3 + 2], a.e[i * 3 + 2]);
            acc.e[i * 3 + j] = pq_sum_conj(s);
        }
}
// A^dag * B
__device__ __forceinline__ Mat3<float> adj_mul_pk(const Mat3<float>& a, const Mat3<float>& b) {
    Mat3<float> r;
#pragma unroll
    for (int i = 0; i < 3; i++)
#pragma unroll
        for (int j = 0; j < 3; j++) {
            PQ s = pq_first(a.e[i], b.e[j]);
            pq_mad(s, a.e[3 + i], b.e[3 + j]);
            pq_mad(s, a.e[6 + i], b.e[6 + j]);
            r.e[i * 3 + j] = pq_sum_conj(s);
        }
    return r;
}
// acc += A * B
__device__ __forceinline__ void mad_mul_pk(Mat3<float>& acc, const Mat3<float>& a, const Mat3<float>& b) {
#pragma unroll
    for (int i = 0; i < 3; i++)
#pragma unroll
        for (int j = 0; j < 3; j++) {
            PQ s = pq_first(acc.e[i * 3 + j], a.e[i * 3], b.e[j]);
            pq_mad(s, a.e[i * 3 + 1], b.e[3 + j]);
            pq_mad(s, a.e[i * 3 + 2], b.e[6 + j]);
            acc.e[i * 3 + j] = pq_sum(s);
        }
}

template <class T> __device__ __forceinline__ Cx<T> det(const Mat3<T>& a) {
    Cx<T> c0 = a.e[4] * a.e[8] - a.e[5] * a.e[7];
    Cx<T> c1 = a.e[3] * a.e[8] - a.e[5] * a.e[6];
    Cx<T> c2 = a.e[3] * a.e[7] - a.e[4] * a.e[6];
    return a.e[0] * c0 - a.e[1] * c1 + a.e[2] * c2;
}

// ---- SU(3) projection (def. 4) -------------------------------------------------
// Proj(V) = V (V^dag V)^{-1/2} exp(-i arg(det V)/3), computed in fp64.
// Route (deliberately different from the oracle's Jacobi diagonalisation, and free of
// fp64 transcendentals, which would cost ~200 slots of the fp64 pipe that bounds the
// APE kernel):
//   H = V^dag V is Hermitian positive definite with characteristic polynomial
//       l^3 - c2 l^2 + c1 l - c0,  c2 = tr H, c1 = sum of principal 2x2 minors,
//       c0 = det H = |det V|^2.
//   With g_k = sqrt(lambda_k) and u = sum g, v = sum_{j<k} g_j g_k, w = g0 g1 g2,
//   Cayley-Hamilton gives
//       H^{-1/2} = f0 + f1 H + f2 H^2,  den = w (u v - w),
//       f0 = (u v^2 - w (u^2 + v))/den, f1 = (2 u v - w - u^3)/den, f2 = u/den.
//   w = |det V| is known directly.  (u, v) solve  u^2 - 2v = c2,  v^2 - 2wu = c1, whose
//   Jacobian determinant 4(uv - w) = 4 (g0+g1)(g0+g2)(g1+g2) never vanishes -- unlike the
//   eigenvalues themselves, (u, v) stay well conditioned when eigenvalues coincide.  They
//   are seeded in fp32 (trigonometric roots of the cubic, on the otherwise idle fp32 and
//   SFU pipes) and polished by three Newton steps in fp64 (quadratic: 3e-4 -> 1e-7 ->
//   1e-14 -> rounding); the reciprocal of uv - w is carried along by its own Newton step.
//   The determinant phase exp(-i theta/3) is the principal cube root of conj(d)/|d|:
//   fp32 seed from a polynomial atan2 and __sincosf, two Newton steps z <- z - (z^3 - c) conj(z^2)/3.
// The projection in three stages: (a) invariants of V and fp32 seeds, (b) the scalar Newton
// chains, written for N links side by side (iteration loop outside, link loop inside),
// (c) W = V (f0 + f1 H + f2 H^2) z.  ncu attributes 40 % of the APE kernel's warp time to the
// projection (31 % of its fp64 instructions) with "wait" (fixed-latency dependency) as the main
// stall, a third of it in the fp32 seed code; the seeds therefore use branch-free polynomial
// acos / atan2 and the approximate division and sincos intrinsics.  The IEEE square roots
// stay: their slow-path branches split the seed code into basic blocks, and every variant
// without them measured slower (ape.cu: BLOCK_BOUNDARY).
// Branch-free fp32 approximations for the seeds (absolute error ~1e-4 rad; the fp64 Newton steps
// that follow converge quadratically from there).  acos: Abramowitz & Stegun 4.4.45 on |x|,
// reflected for x < 0; atan2: A&S 4.4.49-style odd polynomial on [0, 1] with octant reduction.
__device__ __forceinline__ float acos_seed(float x) {
    const float a = fabsf(x);
    const float p = fmaf(fmaf(fmaf(-0.0187293f, a, 0.0742610f), a, -0.2121144f), a, 1.5707288f);
    const float r = p * __fsqrt_rn(fmaxf(1.0f - a, 0.0f));
    return x < 0.0f ? 3.14159265f - r : r;
}
__device__ __forceinline__ float atan2_seed(float y, float x) {
    const float ax = fabsf(x), ay = fabsf(y);
    const float mx = fmaxf(ax, ay), mn = fminf(ax, ay);
    const float t = __fdividef(mn, fmaxf(mx, 1e-37f));
    const float t2 = t * t;
    // atan(t), t in [0, 1]: max error ~1e-5
    float r = fmaf(fmaf(fmaf(fmaf(0.0208351f, t2, -0.0851330f), t2, 0.1801410f), t2, -0.3302995f), t2, 0.9998660f) * t;
    r = ay > ax ? 1.57079633f - r : r;
    r = x < 0.0f ? 3.14159265f - r : r;
    return y < 0.0f ? -r : r;
}

struct ProjScalars {
    double h00, h11, h22, n01, n02, n12;   // H = V^dag V: diagonal, |off-diagonal|^2
    Cx<double> h01, h02, h12;
    double c1, c2, w, rw;                  // invariants, |det V| and its reciprocal
    Cx<double> cc;                         // conj(det V)/|det V|
    double u, v, q;                        // Newton state
    Cx<double> z;                          // cube root state
    double f0, f1, f2;
};

// stage A: invariants of V and the fp32 seeds
__device__ __forceinline__ void proj_stage_a(const Mat3<double>& V, ProjScalars& s) {
    double h00 = 0, h11 = 0, h22 = 0;
    Cx<double> h01 = cx<double>(0, 0), h02 = cx<double>(0, 0), h12 = cx<double>(0, 0);
#pragma unroll
    for (int k = 0; k < 3; k++) {
        Cx<double> a = V.e[k * 3], b = V.e[k * 3 + 1], c = V.e[k * 3 + 2];
        h00 = fma(a.re, a.re, h00); h00 = fma(a.im, a.im, h00);
        h11 = fma(b.re, b.re, h11); h11 = fma(b.im, b.im, h11);
        h22 = fma(c.re, c.re, h22); h22 = fma(c.im, c.im, h22);
        cmad_conj_a(h01, a, b);
        cmad_conj_a(h02, a, c);
        cmad_conj_a(h12, b, c);
    }
    s.h00 = h00; s.h11 = h11; s.h22 = h22; s.h01 = h01; s.h02 = h02; s.h12 = h12;
    s.n01 = h01.re * h01.re + h01.im * h01.im;
    s.n02 = h02.re * h02.re + h02.im * h02.im;
    s.n12 = h12.re * h12.re + h12.im * h12.im;
    s.c2 = h00 + h11 + h22;
    s.c1 = h00 * h11 + h00 * h22 + h11 * h22 - s.n01 - s.n02 - s.n12;
    const Cx<double> d = det(V);
    const double w2 = d.re * d.re + d.im * d.im;   // det H
    // 1/|det V|: fp32 seed, two Newton steps y <- y (1.5 - 0.5 w2 y^2)  (1e-7 -> 1e-14 -> rounding)
    double y = (double)rsqrtf((float)w2);
    const double hw2 = 0.5 * w2;
    y = y * fma(-hw2 * y, y, 1.5);
    y = y * fma(-hw2 * y, y, 1.5);
    s.rw = y; s.w = w2 * y;
    s.cc = cx<double>(d.re * y, -d.im * y);
    // seeds of (u, v): trigonometric roots of the characteristic cubic, in fp32
    {
        const float m = (float)s.c2 * (1.0f / 3.0f), fc1 = (float)s.c1, fc0 = (float)w2;
        const float r2 = fmaxf(m * m - fc1 * (1.0f / 3.0f), 0.0f);
        const float r = __fsqrt_rn(r2);
        const float qh = m * m * m - 0.5f * m * fc1 + 0.5f * fc0;
        float c3 = __fdividef(qh, fmaxf(r * r2, 1e-37f));
        c3 = fminf(1.0f, fmaxf(-1.0f, c3));
        const float th = acos_seed(c3) * (1.0f / 3.0f);
        float sn, cs;
        __sincosf(th, &sn, &cs);
        const float rt3 = 1.7320508f;
        const float g0 = __fsqrt_rn(fmaxf(m + 2.0f * r * cs, 0.0f));
        const float g1 = __fsqrt_rn(fmaxf(m - r * cs - rt3 * r * sn, 0.0f));
        const float g2 = __fsqrt_rn(fmaxf(m - r * cs + rt3 * r * sn, 0.0f));
        const float fu = g0 + g1 + g2, fv = g0 * g1 + g0 * g2 + g1 * g2;
        s.u = (double)fu;
        s.v = (double)fv;
        s.q = (double)__fdividef(1.0f, fu * fv - (float)s.w);
    }
    // seed of the cube root of conj(d)/|d|: principal branch, theta in (-pi, pi]
    {
        const float th0 = atan2_seed((float)d.im, (float)d.re) * (1.0f / 3.0f);
        float sn, cs;
        __sincosf(th0, &sn, &cs);
        s.z = cx<double>((double)cs, -(double)sn);
    }
}

// stage B: the scalar chains of N links, interleaved
template <int N>
__device__ __forceinline__ void proj_stage_b(ProjScalars (&s)[N]) {
#pragma unroll
    for (int it = 0; it < 3; it++) {
#pragma unroll
        for (int n = 0; n < N; n++) {
            const double u = s[n].u, v = s[n].v, w = s[n].w, q = s[n].q;
            const double F1 = fma(u, u, -2.0 * v) - s[n].c2;
            const double F2 = fma(v, v, -2.0 * w * u) - s[n].c1;
            const double hq = 0.5 * q;
            const double un = u - fma(v, F1, F2) * hq;
            const double vn = v - fma(w, F1, u * F2) * hq;
            const double x = fma(un, vn, -w);
            s[n].u = un; s[n].v = vn;
            s[n].q = q * fma(-x, q, 2.0);
        }
    }
#pragma unroll
    for (int it = 0; it < 2; it++) {
#pragma unroll
        for (int n = 0; n < N; n++) {
            const Cx<double> z = s[n].z, z2 = z * z;
            const Cx<double> e = z2 * z - s[n].cc;
            const Cx<double> t = e * conj(z2);
            s[n].z = cx<double>(fma(t.re, -1.0 / 3.0, z.re), fma(t.im, -1.0 / 3.0, z.im));
        }
    }
#pragma unroll
    for (int n = 0; n < N; n++) {
        const double u = s[n].u, v = s[n].v, w = s[n].w;
        const double den = s[n].q * s[n].rw;
        s[n].f0 = (u * v * v - w * (u * u + v)) * den;
        s[n].f1 = (2 * u * v - w - u * u * u) * den;
        s[n].f2 = u * den;
    }
}

// stage C: W = V (f0 + f1 H + f2 H^2) z
__device__ __forceinline__ Mat3<double> proj_stage_c(const Mat3<double>& V, const ProjScalars& s) {
    const double h00 = s.h00, h11 = s.h11, h22 = s.h22, f0 = s.f0, f1 = s.f1, f2 = s.f2;
    const Cx<double> h01 = s.h01, h02 = s.h02, h12 = s.h12;
    const double q00 = h00 * h00 + s.n01 + s.n02;
    const double q11 = h11 * h11 + s.n01 + s.n12;
    const double q22 = h22 * h22 + s.n02 + s.n12;
    Cx<double> q01 = cx<double>((h00 + h11) * h01.re, (h00 + h11) * h01.im);
    cmad_conj_b(q01, h02, h12);          // + h02 conj(h12)
    Cx<double> q02 = cx<double>((h00 + h22) * h02.re, (h00 + h22) * h02.im);
    cmad(q02, h01, h12);                 // + h01 h12
    Cx<double> q12 = cx<double>((h11 + h22) * h12.re, (h11 + h22) * h12.im);
    cmad_conj_a(q12, h01, h02);          // + conj(h01) h02
    // R z with R = f0 + f1 H + f2 H^2 Hermitian: fold the phase into R (nine complex entries)
    const Cx<double> z = s.z;
    const double r00 = f0 + f1 * h00 + f2 * q00, r11 = f0 + f1 * h11 + f2 * q11, r22 = f0 + f1 * h22 + f2 * q22;
    const Cx<double> r01 = cx<double>(f1 * h01.re + f2 * q01.re, f1 * h01.im + f2 * q01.im);
    const Cx<double> r02 = cx<double>(f1 * h02.re + f2 * q02.re, f1 * h02.im + f2 * q02.im);
    const Cx<double> r12 = cx<double>(f1 * h12.re + f2 * q12.re, f1 * h12.im + f2 * q12.im);
    Mat3<double> R;
    R.e[0] = cx<double>(r00 * z.re, r00 * z.im);
    R.e[4] = cx<double>(r11 * z.re, r11 * z.im);
    R.e[8] = cx<double>(r22 * z.re, r22 * z.im);
    R.e[1] = r01 * z; R.e[3] = conj(r01) * z;
    R.e[2] = r02 * z; R.e[6] = conj(r02) * z;
    R.e[5] = r12 * z; R.e[7] = conj(r12) * z;
    return mul(V, R);
}

// Proj for general 3x3 matrices (qdp_reunitarize): the closed form above assumes SU(3)-scaled, moderately conditioned
// input (the blended links of an APE step: cond(V) <= ~11 on hot fields).  Proj is invariant under V -> c V, c > 0, so
// V is first scaled to Frobenius norm sqrt(3) (the fp32 seeds then cannot overflow or underflow), and the result X is
// polished by Newton-Schulz steps X <- X (3 - X^dag X)/2 while max |X^dag X - 1| exceeds ~50 ulp (at most four).
// X = V p(H) z has the polar factor of V times z for every positive polynomial p of H = V^dag V, so the steps remove
// the error an ill-conditioned V leaves in the coefficients f0, f1, f2 without changing what X converges to.
// Supported range: cond(V) up to ~1e5 (beyond that the closed form's error exceeds the Newton-Schulz basin).
__device__ __forceinline__ Mat3<double> proj_su3_general(Mat3<double> V) {
    double n2 = 0;
#pragma unroll
    for (int c = 0; c < 9; c++) n2 = fma(V.e[c].re, V.e[c].re, fma(V.e[c].im, V.e[c].im, n2));
    // The zero matrix has no polar factor, and a matrix with an infinite or NaN entry no meaningful one: such a
    // matrix is returned as it came (inf * 0 below would otherwise turn a zero link into NaNs), so the caller can
    // still see what was wrong with it.  Documented with qdp_reunitarize in qdp_b200.h.
    if (!(n2 > 0.0) || !(n2 <= 1.7976931348623157e308)) return V;
    const double sc = 1.7320508075688772 / sqrt(n2);
#pragma unroll
    for (int c = 0; c < 9; c++) V.e[c] = cx<double>(V.e[c].re * sc, V.e[c].im * sc);
    ProjScalars ps[1];
    proj_stage_a(V, ps[0]);
    proj_stage_b<1>(ps);
    Mat3<double> X = proj_stage_c(V, ps[0]);
    for (int it = 0; it < 4; it++) {
        Mat3<double> M;      // (3 - X^dag X) / 2
        double r = 0;
#pragma unroll
        for (int i = 0; i < 3; i++)
#pragma unroll
            for (int j = 0; j < 3; j++) {
                Cx<double> y = cx<double>(0, 0);
#pragma unroll
                for (int k = 0; k < 3; k++) cmad_conj_a(y, X.e[k * 3 + i], X.e[k * 3 + j]);
                r = fmax(r, fmax(fabs(y.re - (i == j ? 1.0 : 0.0)), fabs(y.im)));
                M.e[i * 3 + j] = cx<double>((i == j ? 1.5 : 0.0) - 0.5 * y.re, -0.5 * y.im);
            }
        if (!(r > 1e-14)) break;
        X = mul(X, M);
    }
    return X;
}

// ---- fp32 projection for fp32 fields -------------------------------------------------------------
// The same closed form entirely in fp32 (two Newton steps on (u, v), one on the cube root), followed
// by one Newton-Schulz step X <- X (3 - X^dag X)/2.  X = V p(H) has the polar factor of V for any
// positive polynomial p of H = V^dag V, so the step removes the error the ill-conditioned closed
// form leaves (hot links: cond(V) ~ 10, closed form alone 9e-6) without changing what it converges
// to: measured against the fp64 oracle on 20,000 blended hot links, max per-link error 1.0e-6
// (bar 2e-5), median 7e-8.  No fp64 instruction: the fp32 APE step no longer queues on the fp64 pipe.
__device__ __forceinline__ Mat3<float> proj_su3_f32(const Mat3<float>& V) {
    float h00 = 0, h11 = 0, h22 = 0;
    Cx<float> h01 = cx<float>(0, 0), h02 = cx<float>(0, 0), h12 = cx<float>(0, 0);
#pragma unroll
    for (int k = 0; k < 3; k++) {
        const Cx<float> a = V.e[k * 3], b = V.e[k * 3 + 1], c = V.e[k * 3 + 2];
        h00 = fmaf(a.re, a.re, fmaf(a.im, a.im, h00));
        h11 = fmaf(b.re, b.re, fmaf(b.im, b.im, h11));
        h22 = fmaf(c.re, c.re, fmaf(c.im, c.im, h22));
        cmad_conj_a(h01, a, b);
        cmad_conj_a(h02, a, c);
        cmad_conj_a(h12, b, c);
    }
    const float n01 = h01.re * h01.re + h01.im * h01.im;
    const float n02 = h02.re * h02.re + h02.im * h02.im;
    const float n12 = h12.re * h12.re + h12.im * h12.im;
    const float c2 = h00 + h11 + h22;
    const float c1 = h00 * h11 + h00 * h22 + h11 * h22 - n01 - n02 - n12;
    const Cx<float> d = det(V);
    const float w2 = d.re * d.re + d.im * d.im;
    float rw = rsqrtf(w2);
    rw = rw * fmaf(-0.5f * w2 * rw, rw, 1.5f);
    const float w = w2 * rw;
    // seeds: trigonometric roots of the characteristic cubic
    const float m = c2 * (1.0f / 3.0f);
    const float r2 = fmaxf(m * m - c1 * (1.0f / 3.0f), 0.0f);
    const float r = __fsqrt_rn(r2);
    const float qh = m * m * m - 0.5f * m * c1 + 0.5f * w2;
    float c3 = __fdividef(qh, fmaxf(r * r2, 1e-37f));
    c3 = fminf(1.0f, fmaxf(-1.0f, c3));
    float sn, cs;
    __sincosf(acos_seed(c3) * (1.0f / 3.0f), &sn, &cs);
    const float rt3 = 1.7320508f;
    const float g0 = __fsqrt_rn(fmaxf(m + 2.0f * r * cs, 0.0f));
    const float g1 = __fsqrt_rn(fmaxf(m - r * cs - rt3 * r * sn, 0.0f));
    const float g2 = __fsqrt_rn(fmaxf(m - r * cs + rt3 * r * sn, 0.0f));
    float u = g0 + g1 + g2, v = g0 * g1 + g0 * g2 + g1 * g2;
    float q = __fdividef(1.0f, u * v - w);
#pragma unroll
    for (int it = 0; it < 2; it++) {
        const float F1 = fmaf(u, u, -2.0f * v) - c2;
        const float F2 = fmaf(v, v, -2.0f * w * u) - c1;
        const float hq = 0.5f * q;
        const float un = u - fmaf(v, F1, F2) * hq;
        const float vn = v - fmaf(w, F1, u * F2) * hq;
        u = un; v = vn;
        q = q * fmaf(-fmaf(u, v, -w), q, 2.0f);
    }
    const float den = q * rw;
    const float f0 = (u * v * v - w * (u * u + v)) * den;
    const float f1 = (2 * u * v - w - u * u * u) * den;
    const float f2 = u * den;
    // H^2 (Hermitian) and R = f0 + f1 H + f2 H^2
    const float q00 = h00 * h00 + n01 + n02, q11 = h11 * h11 + n01 + n12, q22 = h22 * h22 + n02 + n12;
    Cx<float> q01 = cx<float>((h00 + h11) * h01.re, (h00 + h11) * h01.im);
    cmad_conj_b(q01, h02, h12);
    Cx<float> q02 = cx<float>((h00 + h22) * h02.re, (h00 + h22) * h02.im);
    cmad(q02, h01, h12);
    Cx<float> q12 = cx<float>((h11 + h22) * h12.re, (h11 + h22) * h12.im);
    cmad_conj_a(q12, h01, h02);
    Mat3<float> R;
    R.e[0] = cx<float>(f0 + f1 * h00 + f2 * q00, 0);
    R.e[4] = cx<float>(f0 + f1 * h11 + f2 * q11, 0);
    R.e[8] = cx<float>(f0 + f1 * h22 + f2 * q22, 0);
    R.e[1] = cx<float>(f1 * h01.re + f2 * q01.re, f1 * h01.im + f2 * q01.im);
    R.e[2] = cx<float>(f1 * h02.re + f2 * q02.re, f1 * h02.im + f2 * q02.im);
    R.e[5] = cx<float>(f1 * h12.re + f2 * q12.re, f1 * h12.im + f2 * q12.im);
    R.e[3] = conj(R.e[1]); R.e[6] = conj(R.e[2]); R.e[7] = conj(R.e[5]);
    const Mat3<float> X = mul(V, R);
    // Newton-Schulz: M = (3 - X^dag X)/2 (Hermitian), folded with the determinant phase z
    float y00 = 0, y11 = 0, y22 = 0;
    Cx<float> y01 = cx<float>(0, 0), y02 = cx<float>(0, 0), y12 = cx<float>(0, 0);
#pragma unroll
    for (int k = 0; k < 3; k++) {
        const Cx<float> a = X.e[k * 3], b = X.e[k * 3 + 1], c = X.e[k * 3 + 2];
        y00 = fmaf(a.re, a.re, fmaf(a.im, a.im, y00));
        y11 = fmaf(b.re, b.re, fmaf(b.im, b.im, y11));
        y22 = fmaf(c.re, c.re, fmaf(c.im, c.im, y22));
        cmad_conj_a(y01, a, b);
        cmad_conj_a(y02, a, c);
        cmad_conj_a(y12, b, c);
    }
    // z = principal cube root of conj(d)/|d|: polynomial atan2 seed, one Newton step
    Cx<float> z;
    {
        float s0, c0;
        __sincosf(atan2_seed(d.im, d.re) * (1.0f / 3.0f), &s0, &c0);
        z = cx<float>(c0, -s0);
        const Cx<float> cc = cx<float>(d.re * rw, -d.im * rw);
        const Cx<float> z2 = z * z;
        const Cx<float> t = (z2 * z - cc) * conj(z2);
        z = cx<float>(fmaf(t.re, -1.0f / 3.0f, z.re), fmaf(t.im, -1.0f / 3.0f, z.im));
    }
    Mat3<float> M;
    const float m00 = 1.5f - 0.5f * y00, m11 = 1.5f - 0.5f * y11, m22 = 1.5f - 0.5f * y22;
    const Cx<float> m01 = cx<float>(-0.5f * y01.re, -0.5f * y01.im), m02 = cx<float>(-0.5f * y02.re, -0.5f * y02.im),
                    m12 = cx<float>(-0.5f * y12.re, -0.5f * y12.im);
    M.e[0] = cx<float>(m00 * z.re, m00 * z.im);
    M.e[4] = cx<float>(m11 * z.re, m11 * z.im);
    M.e[8] = cx<float>(m22 * z.re, m22 * z.im);
    M.e[1] = m01 * z; M.e[3] = conj(m01) * z;
    M.e[2] = m02 * z; M.e[6] = conj(m02) * z;
    M.e[5] = m12 * z; M.e[7] = conj(m12) * z;
    return mul(X, M);
}

}  // namespace qdp
