// su3.cuh -- per-site colour algebra in registers: 3x3 complex matrices, colour
// vectors, field loads/stores in the site-fastest SoA layout, and the SU(3)
// projection.  (8(c) definitions 2-5.)
//
// Device field layout: component plane c holds V complex
// numbers, dev[c*V + s], s the internal site index, complex = (re, im) adjacent:
// fp64 -> one double2 = one 128-bit access per thread, a warp moves 512
// contiguous bytes per plane; fp32 -> float2, 256 contiguous bytes per warp.
#pragma once
#include <cuda_runtime.h>

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
__device__ __forceinline__ T2* site_ptr(T2* f, int ncomp, int c0, int s) {
    return f + ((size_t)(s >> 5) * ncomp + c0) * kLane + (s & 31);
}
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
// colour matrix number `m` of a field with ncomp components (gauge: 36, m = mu; colour matrix: 9, m = 0)
template <class T>
__device__ __forceinline__ Mat3<T> ld_mat(const typename Vec2<T>::type* __restrict__ f, int ncomp, int m, int s) {
    return ld_mat_at<T>(site_ptr(f, ncomp, m * 9, s));
}
template <class T>
__device__ __forceinline__ Spinor<T> ld_spinor(const typename Vec2<T>::type* __restrict__ f, int s) {
    const typename Vec2<T>::type* p = site_ptr(f, 12, 0, s);
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
// Re tr(A * B^dag) = sum_ij Re(A_ij conj(B_ij))
template <class T> __device__ __forceinline__ T re_tr_mul_adj(const Mat3<T>& a, const Mat3<T>& b) {
    T s = 0;
#pragma unroll
    for (int i = 0; i < 9; i++) { s = fma(a.e[i].re, b.e[i].re, s); s = fma(a.e[i].im, b.e[i].im, s); }
    return s;
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
//   fp32 seed from atan2f/sincosf, two Newton steps z <- z - (z^3 - c) conj(z^2)/3.
__device__ __forceinline__ Mat3<double> proj_su3(const Mat3<double>& V) {
    // H = V^dag V: diagonal real, upper triangle complex
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
    const double n01 = h01.re * h01.re + h01.im * h01.im;
    const double n02 = h02.re * h02.re + h02.im * h02.im;
    const double n12 = h12.re * h12.re + h12.im * h12.im;
    const double c2 = h00 + h11 + h22;
    const double c1 = h00 * h11 + h00 * h22 + h11 * h22 - n01 - n02 - n12;
    const Cx<double> d = det(V);
    const double w2 = d.re * d.re + d.im * d.im;   // det H
    const double rw = rsqrt(w2), w = w2 * rw;      // 1/|det V|, |det V|
    // ---- fp32 seeds ----
    double u, v, q;
    {
        const float m = (float)c2 * (1.0f / 3.0f), fc1 = (float)c1, fc0 = (float)w2;
        const float r2 = fmaxf(m * m - fc1 * (1.0f / 3.0f), 0.0f);
        const float r = sqrtf(r2);
        const float qh = m * m * m - 0.5f * m * fc1 + 0.5f * fc0;
        float c3 = qh / fmaxf(r * r2, 1e-37f);
        c3 = fminf(1.0f, fmaxf(-1.0f, c3));
        const float th = acosf(c3) * (1.0f / 3.0f);
        float s, c;
        __sincosf(th, &s, &c);
        const float rt3 = 1.7320508f;
        const float g0 = sqrtf(fmaxf(m + 2.0f * r * c, 0.0f));
        const float g1 = sqrtf(fmaxf(m - r * c - rt3 * r * s, 0.0f));
        const float g2 = sqrtf(fmaxf(m - r * c + rt3 * r * s, 0.0f));
        const float fu = g0 + g1 + g2, fv = g0 * g1 + g0 * g2 + g1 * g2;
        u = (double)fu;
        v = (double)fv;
        q = (double)(1.0f / (fu * fv - (float)w));
    }
    // ---- Newton on (u, v), q -> 1/(uv - w) ----
#pragma unroll
    for (int it = 0; it < 3; it++) {
        const double F1 = fma(u, u, -2.0 * v) - c2;
        const double F2 = fma(v, v, -2.0 * w * u) - c1;
        const double hq = 0.5 * q;
        const double du = fma(v, F1, F2) * hq;
        const double dv = fma(w, F1, u * F2) * hq;
        u -= du;
        v -= dv;
        const double x = fma(u, v, -w);
        q = q * fma(-x, q, 2.0);
    }
    const double den = q * rw;
    const double f0 = (u * v * v - w * (u * u + v)) * den;
    const double f1 = (2 * u * v - w - u * u * u) * den;
    const double f2 = u * den;
    // H^2 (Hermitian): diagonal and upper triangle
    const double q00 = h00 * h00 + n01 + n02;
    const double q11 = h11 * h11 + n01 + n12;
    const double q22 = h22 * h22 + n02 + n12;
    Cx<double> q01 = cx<double>((h00 + h11) * h01.re, (h00 + h11) * h01.im);
    cmad_conj_b(q01, h02, h12);          // + h02 conj(h12)
    Cx<double> q02 = cx<double>((h00 + h22) * h02.re, (h00 + h22) * h02.im);
    cmad(q02, h01, h12);                 // + h01 h12
    Cx<double> q12 = cx<double>((h11 + h22) * h12.re, (h11 + h22) * h12.im);
    cmad_conj_a(q12, h01, h02);          // + conj(h01) h02
    // R = f0 + f1 H + f2 H^2 (Hermitian)
    Mat3<double> R;
    R.e[0] = cx<double>(f0 + f1 * h00 + f2 * q00, 0);
    R.e[4] = cx<double>(f0 + f1 * h11 + f2 * q11, 0);
    R.e[8] = cx<double>(f0 + f1 * h22 + f2 * q22, 0);
    R.e[1] = cx<double>(f1 * h01.re + f2 * q01.re, f1 * h01.im + f2 * q01.im);
    R.e[2] = cx<double>(f1 * h02.re + f2 * q02.re, f1 * h02.im + f2 * q02.im);
    R.e[5] = cx<double>(f1 * h12.re + f2 * q12.re, f1 * h12.im + f2 * q12.im);
    R.e[3] = conj(R.e[1]); R.e[6] = conj(R.e[2]); R.e[7] = conj(R.e[5]);
    Mat3<double> W = mul(V, R);
    // ---- determinant phase: z = principal cube root of conj(d)/|d| (arg det W = arg det V since R > 0) ----
    Cx<double> z;
    {
        const float th0 = atan2f((float)d.im, (float)d.re) * (1.0f / 3.0f);
        float s, c;
        sincosf(th0, &s, &c);
        z = cx<double>((double)c, -(double)s);
    }
    const Cx<double> cc = cx<double>(d.re * rw, -d.im * rw);
#pragma unroll
    for (int it = 0; it < 2; it++) {
        const Cx<double> z2 = z * z;
        const Cx<double> e = z2 * z - cc;
        const Cx<double> t = e * conj(z2);
        z.re = fma(t.re, -1.0 / 3.0, z.re);
        z.im = fma(t.im, -1.0 / 3.0, z.im);
    }
#pragma unroll
    for (int i = 0; i < 9; i++) W.e[i] = W.e[i] * z;
    return W;
}

}  // namespace qdp
