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
template <class T>
__device__ __forceinline__ Cx<T> ld_cx(const typename Vec2<T>::type* __restrict__ f, size_t V, int c, int s) {
    typename Vec2<T>::type v = __ldg(f + (size_t)c * V + s);
    return cx<T>(v.x, v.y);
}
template <class T>
__device__ __forceinline__ void st_cx(typename Vec2<T>::type* __restrict__ f, size_t V, int c, int s, Cx<T> v) {
    typename Vec2<T>::type o;
    o.x = v.re; o.y = v.im;
    f[(size_t)c * V + s] = o;
}
// colour matrix number `m` of a field (gauge: m = mu; colour-matrix field: m = 0)
template <class T>
__device__ __forceinline__ Mat3<T> ld_mat(const typename Vec2<T>::type* __restrict__ f, size_t V, int m, int s) {
    Mat3<T> r;
#pragma unroll
    for (int c = 0; c < 9; c++) r.e[c] = ld_cx<T>(f, V, m * 9 + c, s);
    return r;
}
template <class T>
__device__ __forceinline__ void st_mat(typename Vec2<T>::type* __restrict__ f, size_t V, int m, int s, const Mat3<T>& a) {
#pragma unroll
    for (int c = 0; c < 9; c++) st_cx<T>(f, V, m * 9 + c, s, a.e[c]);
}
template <class T>
__device__ __forceinline__ Spinor<T> ld_spinor(const typename Vec2<T>::type* __restrict__ f, size_t V, int s) {
    Spinor<T> r;
#pragma unroll
    for (int c = 0; c < 12; c++) r.e[c] = ld_cx<T>(f, V, c, s);
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
// Proj(V) = V (V^dag V)^{-1/2} exp(-i arg(det V)/3).
// Route (deliberately different from the oracle's Jacobi diagonalisation):
//   H = V^dag V is Hermitian positive definite.  Its eigenvalues come from the
//   trigonometric solution of the characteristic cubic of K = H - (tr H/3) 1:
//       lambda_k = m + 2 r cos(theta + 2 pi k/3), r^2 = tr K^2 / 6,
//       cos 3 theta = det K / (2 r^3).
//   With g_k = sqrt(lambda_k) and the symmetric functions u = sum g, v = sum g g',
//   w = g0 g1 g2, Cayley-Hamilton gives
//       H^{-1/2} = f0 + f1 H + f2 H^2,  den = w (u v - w),
//       f0 = (u v^2 - w (u^2 + v))/den, f1 = (2 u v - w - u^3)/den, f2 = u/den.
//   The three roots always have the exact sum 3m and exact sum of squares, so an
//   error in theta only perturbs det: the root set is backward stable even when
//   two eigenvalues nearly coincide, and f0, f1, f2 are smooth symmetric functions.
template <class T> __device__ __forceinline__ Mat3<T> proj_su3(const Mat3<T>& V) {
    // H = V^dag V: diagonal real, upper triangle complex
    T h00 = 0, h11 = 0, h22 = 0;
    Cx<T> h01 = cx<T>(0, 0), h02 = cx<T>(0, 0), h12 = cx<T>(0, 0);
#pragma unroll
    for (int k = 0; k < 3; k++) {
        Cx<T> a = V.e[k * 3], b = V.e[k * 3 + 1], c = V.e[k * 3 + 2];
        h00 = fma(a.re, a.re, h00); h00 = fma(a.im, a.im, h00);
        h11 = fma(b.re, b.re, h11); h11 = fma(b.im, b.im, h11);
        h22 = fma(c.re, c.re, h22); h22 = fma(c.im, c.im, h22);
        cmad_conj_a(h01, a, b);
        cmad_conj_a(h02, a, c);
        cmad_conj_a(h12, b, c);
    }
    T n01 = h01.re * h01.re + h01.im * h01.im;
    T n02 = h02.re * h02.re + h02.im * h02.im;
    T n12 = h12.re * h12.re + h12.im * h12.im;
    T m = (h00 + h11 + h22) / T(3);
    T k00 = h00 - m, k11 = h11 - m, k22 = h22 - m;
    T r2 = (k00 * k00 + k11 * k11 + k22 * k22) * T(1.0 / 6.0) + (n01 + n02 + n12) * T(1.0 / 3.0);
    T l0, l1, l2;
    if (r2 <= T(1e-30) * m * m) {       // H = m * 1 (e.g. V a multiple of a unitary matrix)
        l0 = l1 = l2 = m;
    } else {
        T r = sqrt(r2);
        // det K, K Hermitian
        Cx<T> t = h01 * h12;            // k01 k12
        T re3 = t.re * h02.re + t.im * h02.im;   // Re(k01 k12 conj(k02))
        T dK = k00 * (k11 * k22 - n12) - k22 * n01 - k11 * n02 + 2 * re3;
        T c3 = dK / (2 * r * r2);
        c3 = fmin(T(1), fmax(T(-1), c3));
        T th = acos(c3) * T(1.0 / 3.0);
        T s, c;
        sincos(th, &s, &c);
        const T rt3 = T(1.7320508075688772935);
        l0 = m + 2 * r * c;
        l1 = m - r * c - rt3 * r * s;
        l2 = m - r * c + rt3 * r * s;
    }
    T g0 = sqrt(l0), g1 = sqrt(l1), g2 = sqrt(l2);
    T u = g0 + g1 + g2, v = g0 * g1 + g0 * g2 + g1 * g2, w = g0 * g1 * g2;
    T den = T(1) / (w * (u * v - w));
    T f0 = (u * v * v - w * (u * u + v)) * den;
    T f1 = (2 * u * v - w - u * u * u) * den;
    T f2 = u * den;
    // H^2 (Hermitian): diagonal and upper triangle
    T q00 = h00 * h00 + n01 + n02;
    T q11 = h11 * h11 + n01 + n12;
    T q22 = h22 * h22 + n02 + n12;
    Cx<T> q01 = cx<T>((h00 + h11) * h01.re, (h00 + h11) * h01.im);
    cmad_conj_b(q01, h02, h12);          // + h02 conj(h12)
    Cx<T> q02 = cx<T>((h00 + h22) * h02.re, (h00 + h22) * h02.im);
    cmad(q02, h01, h12);                 // + h01 h12
    Cx<T> q12 = cx<T>((h11 + h22) * h12.re, (h11 + h22) * h12.im);
    cmad_conj_a(q12, h01, h02);          // + conj(h01) h02
    // R = f0 + f1 H + f2 H^2 (Hermitian)
    Mat3<T> R;
    R.e[0] = cx<T>(f0 + f1 * h00 + f2 * q00, 0);
    R.e[4] = cx<T>(f0 + f1 * h11 + f2 * q11, 0);
    R.e[8] = cx<T>(f0 + f1 * h22 + f2 * q22, 0);
    R.e[1] = cx<T>(f1 * h01.re + f2 * q01.re, f1 * h01.im + f2 * q01.im);
    R.e[2] = cx<T>(f1 * h02.re + f2 * q02.re, f1 * h02.im + f2 * q02.im);
    R.e[5] = cx<T>(f1 * h12.re + f2 * q12.re, f1 * h12.im + f2 * q12.im);
    R.e[3] = conj(R.e[1]); R.e[6] = conj(R.e[2]); R.e[7] = conj(R.e[5]);
    Mat3<T> W = mul(V, R);
    // remove the determinant phase: arg det W = arg det V since R > 0
    Cx<T> d = det(V);
    T theta = atan2(d.im, d.re) * T(1.0 / 3.0);
    T ps, pc;
    sincos(theta, &ps, &pc);
    Cx<T> ph = cx<T>(pc, -ps);
#pragma unroll
    for (int i = 0; i < 9; i++) W.e[i] = W.e[i] * ph;
    return W;
}

}  // namespace qdp
