// expr.cuh -- a compile-time expression layer: lattice expressions written the way they look on paper become ONE
// kernel each, evaluated site by site without temporaries.
//
// This is the paper's contribution restated for the device: QDP++ builds PETE expression templates and the paper's
// tree parser turns each tree into one generated CUDA kernel.  Here the tree is a C++
// type, its leaves are field operands, and nvcc instantiates the kernel at build time (no JIT): the expression
//
//     sum(real(trace(u[mu] * shift(u[nu], mu) * adj(shift(u[mu], nu)) * adj(u[nu]))))
//
// is written below as  real(trace(U<MU>() * shift<MU,+1>(U<NU>()) * adj(shift<NU,+1>(U<MU>())) * adj(U<NU>())))
// and handed to sum2_kernel.  Leaves:  M<ARG,NCOMP,SLOT> (matrix SLOT of field operand ARG), Mrt<ARG> (slot chosen at
// run time), F<ARG> (fermion field operand ARG), Sc<K> (real scalar operand K).  Nodes:  a * b, a + b, adj(a), trace(a), real(a), shift<MU,SIGN>(a) and
// shift_rt(a) -- a shift moves the evaluation point of its whole sub-expression, so shift<NU,-1>(adj(U<NU>()) *
// U<MU>() * shift<MU,+1>(U<NU>())) is the lower staple with its two-hop leaf.  trace(a * b) and real(trace(a * b)) are
// evaluated without forming the product (9 complex / 18 real multiply-adds).  Assignment under a subset:
// assign_kernel (matrix- or complex-valued expression -> field slot); fused global sums: sum2_kernel.
#pragma once
#ifndef __CUDACC_RTC__
#include <type_traits>

#include "internal.h"
#endif
#include "reduce.cuh"
#include "su3.cuh"

namespace qdp {
namespace ex {

struct Args {
    const void* f[4];   // field operands (device pointers, the element type is the kernel's precision)
    int ncomp[4];       // components per site of each operand (9 colour matrix, 36 gauge)
    int slot[4];        // run-time matrix number for Mrt leaves
    int mu, sign;       // run-time direction for shift_rt; mu < 0: no shift
    double sc[4];       // real scalars
};

template <class T> struct Env {
    const Geom& g;
    Site x;             // where the (sub-)expression is evaluated
    const Args& a;
};

struct Node {};
#ifndef __CUDACC_RTC__
template <class E> constexpr bool is_node = std::is_base_of<Node, E>::value;
#endif

// ---- values and their arithmetic ------------------------------------------------------------
template <class T> __device__ __forceinline__ Mat3<T> v_adj(const Mat3<T>& a) {
    Mat3<T> r;
#pragma unroll
    for (int i = 0; i < 3; i++)
#pragma unroll
        for (int j = 0; j < 3; j++) r.e[i * 3 + j] = conj(a.e[j * 3 + i]);
    return r;
}
template <class T> __device__ __forceinline__ Cx<T> v_adj(const Cx<T>& a) { return conj(a); }
template <class T> __device__ __forceinline__ T v_adj(T a) { return a; }

template <class T> __device__ __forceinline__ Mat3<T> v_mul(const Mat3<T>& a, const Mat3<T>& b) { return mul(a, b); }
template <class T> __device__ __forceinline__ Mat3<T> v_mul(T s, const Mat3<T>& b) {
    Mat3<T> r;
#pragma unroll
    for (int i = 0; i < 9; i++) r.e[i] = cx<T>(s * b.e[i].re, s * b.e[i].im);
    return r;
}
template <class T> __device__ __forceinline__ Mat3<T> v_mul(const Mat3<T>& b, T s) { return v_mul(s, b); }
template <class T> __device__ __forceinline__ Cx<T> v_mul(Cx<T> a, Cx<T> b) { return a * b; }
template <class T> __device__ __forceinline__ Cx<T> v_mul(T s, Cx<T> b) { return cx<T>(s * b.re, s * b.im); }
template <class T> __device__ __forceinline__ T v_mul(T a, T b) { return a * b; }

template <class T> __device__ __forceinline__ Mat3<T> v_add(const Mat3<T>& a, const Mat3<T>& b) {
    Mat3<T> r;
#pragma unroll
    for (int i = 0; i < 9; i++) r.e[i] = a.e[i] + b.e[i];
    return r;
}
template <class T> __device__ __forceinline__ Cx<T> v_add(Cx<T> a, Cx<T> b) { return a + b; }
template <class T> __device__ __forceinline__ T v_add(T a, T b) { return a + b; }

// spin-colour vectors (fermions): a colour matrix rotates the colour index of each spin component (the hopping term's product)
template <class T> __device__ __forceinline__ Spinor<T> v_mul(const Mat3<T>& u, const Spinor<T>& p) {
    Spinor<T> r;
#pragma unroll
    for (int sp = 0; sp < 4; sp++)
#pragma unroll
        for (int a = 0; a < 3; a++) {
            Cx<T> s = u.e[a * 3] * p.e[sp * 3];
            cmad(s, u.e[a * 3 + 1], p.e[sp * 3 + 1]);
            cmad(s, u.e[a * 3 + 2], p.e[sp * 3 + 2]);
            r.e[sp * 3 + a] = s;
        }
    return r;
}
template <class T> __device__ __forceinline__ Spinor<T> v_mul(T s, const Spinor<T>& p) {
    Spinor<T> r;
#pragma unroll
    for (int i = 0; i < 12; i++) r.e[i] = cx<T>(s * p.e[i].re, s * p.e[i].im);
    return r;
}
template <class T> __device__ __forceinline__ Spinor<T> v_mul(const Spinor<T>& p, T s) { return v_mul(s, p); }
template <class T> __device__ __forceinline__ Spinor<T> v_mul(Cx<T> z, const Spinor<T>& p) {
    Spinor<T> r;
#pragma unroll
    for (int i = 0; i < 12; i++) r.e[i] = z * p.e[i];
    return r;
}
template <class T> __device__ __forceinline__ Spinor<T> v_add(const Spinor<T>& a, const Spinor<T>& b) {
    Spinor<T> r;
#pragma unroll
    for (int i = 0; i < 12; i++) r.e[i] = a.e[i] + b.e[i];
    return r;
}
// site-local norm and inner product (QDP++ localNorm2 / localInnerProduct): sum over spin and colour
template <class T> __device__ __forceinline__ T v_norm2(const Spinor<T>& a) {
    T s = 0;
#pragma unroll
    for (int i = 0; i < 12; i++) { s = fma(a.e[i].re, a.e[i].re, s); s = fma(a.e[i].im, a.e[i].im, s); }
    return s;
}
template <class T> __device__ __forceinline__ Cx<T> v_inner(const Spinor<T>& a, const Spinor<T>& b) {
    Cx<T> s = cx<T>(0, 0);
#pragma unroll
    for (int i = 0; i < 12; i++) cmad_conj_a(s, a.e[i], b.e[i]);
    return s;
}

template <class T> __device__ __forceinline__ Mat3<T> v_neg(const Mat3<T>& a) {
    Mat3<T> r;
#pragma unroll
    for (int i = 0; i < 9; i++) r.e[i] = cx<T>(-a.e[i].re, -a.e[i].im);
    return r;
}
template <class T> __device__ __forceinline__ Spinor<T> v_neg(const Spinor<T>& a) {
    Spinor<T> r;
#pragma unroll
    for (int i = 0; i < 12; i++) r.e[i] = cx<T>(-a.e[i].re, -a.e[i].im);
    return r;
}
template <class T> __device__ __forceinline__ Cx<T> v_neg(Cx<T> a) { return cx<T>(-a.re, -a.im); }
template <class T> __device__ __forceinline__ T v_neg(T a) { return -a; }

template <class T> __device__ __forceinline__ Cx<T> v_trace(const Mat3<T>& a) { return a.e[0] + a.e[4] + a.e[8]; }
template <class T> __device__ __forceinline__ T v_real(Cx<T> a) { return a.re; }
template <class T> __device__ __forceinline__ T v_imag(Cx<T> a) { return a.im; }

// ---- leaves -------------------------------------------------------------------------------------
template <int ARG, int NCOMP, int SLOT> struct M : Node {
    template <class T> __device__ __forceinline__ static Mat3<T> eval(const Env<T>& e) {
        using T2 = typename Vec2<T>::type;
        const Geom& g = e.g;
        return ld_mat_at<T>(site_ptr(static_cast<const T2*>(e.a.f[ARG]), NCOMP, SLOT * 9, e.x.index(g)));
    }
};
template <int ARG> struct Mrt : Node {
    template <class T> __device__ __forceinline__ static Mat3<T> eval(const Env<T>& e) {
        using T2 = typename Vec2<T>::type;
        const Geom& g = e.g;
        return ld_mat_at<T>(site_ptr(static_cast<const T2*>(e.a.f[ARG]), e.a.ncomp[ARG], e.a.slot[ARG] * 9, e.x.index(g)));
    }
};
template <int ARG> struct F : Node {   // fermion field operand ARG
    template <class T> __device__ __forceinline__ static Spinor<T> eval(const Env<T>& e) {
        using T2 = typename Vec2<T>::type;
        const Geom& g = e.g;
        return ld_spinor_at<T>(site_ptr(static_cast<const T2*>(e.a.f[ARG]), 12, 0, e.x.index(g)));
    }
};
template <int K> struct Sc : Node {
    template <class T> __device__ __forceinline__ static T eval(const Env<T>& e) { return (T)e.a.sc[K]; }
};
template <int SLOT> using U = M<0, 36, SLOT>;   // link SLOT of a gauge field in operand 0

// ---- nodes ---------------------------------------------------------------------------------------
template <class E, int MU, int SIGN> struct Shifted : Node {
    template <class T> __device__ __forceinline__ static auto eval(const Env<T>& e) {
        const Env<T> n{e.g, site_step<MU, SIGN>(e.g, e.x), e.a};
        return E::template eval<T>(n);
    }
};
template <class E> struct ShiftedRt : Node {
    template <class T> __device__ __forceinline__ static auto eval(const Env<T>& e) {
        const Env<T> n{e.g, e.a.mu < 0 ? e.x : site_step_rt(e.g, e.x, e.a.mu, e.a.sign), e.a};
        return E::template eval<T>(n);
    }
};
template <class E> struct Adjoint : Node {
    template <class T> __device__ __forceinline__ static auto eval(const Env<T>& e) { return v_adj(E::template eval<T>(e)); }
};
template <class A, class B> struct Product : Node {
    template <class T> __device__ __forceinline__ static auto eval(const Env<T>& e) {
        return v_mul(A::template eval<T>(e), B::template eval<T>(e));
    }
};
template <class A, class B> struct Sum : Node {
    template <class T> __device__ __forceinline__ static auto eval(const Env<T>& e) {
        return v_add(A::template eval<T>(e), B::template eval<T>(e));
    }
};
// -e, and a - b = a + (-b) (exactly the IEEE difference)
template <class E> struct Neg : Node {
    template <class T> __device__ __forceinline__ static auto eval(const Env<T>& e) { return v_neg(E::template eval<T>(e)); }
};
template <class A, class B> struct Diff : Node {
    template <class T> __device__ __forceinline__ static auto eval(const Env<T>& e) {
        return v_add(A::template eval<T>(e), v_neg(B::template eval<T>(e)));
    }
};
// a real literal, carried in the type as the bit pattern of the double (cast to the field precision like a scalar argument)
template <unsigned long long BITS> struct Lit : Node {
    template <class T> __device__ __forceinline__ static T eval(const Env<T>&) { return (T)__longlong_as_double((long long)BITS); }
};
template <class E> struct Trace : Node {
    template <class T> __device__ __forceinline__ static Cx<T> eval(const Env<T>& e) { return v_trace(E::template eval<T>(e)); }
};
// trace(a * b) = sum_ij a_ij b_ji: no product is formed when both factors are matrices; any other pair the
// language allows under a trace (real scalar * matrix, either order) takes the plain route
template <class T> __device__ __forceinline__ Cx<T> v_trace_mul(const Mat3<T>& a, const Mat3<T>& b) {
    Cx<T> s = cx<T>(0, 0);
#pragma unroll
    for (int i = 0; i < 3; i++)
#pragma unroll
        for (int j = 0; j < 3; j++) cmad(s, a.e[i * 3 + j], b.e[j * 3 + i]);
    return s;
}
template <class T> __device__ __forceinline__ Cx<T> v_trace_mul(T s, const Mat3<T>& b) { return v_mul(s, v_trace(b)); }
template <class T> __device__ __forceinline__ Cx<T> v_trace_mul(const Mat3<T>& a, T s) { return v_mul(s, v_trace(a)); }
template <class A, class B> struct Trace<Product<A, B>> : Node {
    template <class T> __device__ __forceinline__ static Cx<T> eval(const Env<T>& e) {
        return v_trace_mul(A::template eval<T>(e), B::template eval<T>(e));
    }
};
template <class E> struct Real : Node {
    template <class T> __device__ __forceinline__ static T eval(const Env<T>& e) { return v_real(E::template eval<T>(e)); }
};
// real(trace(a * b)) = sum_ij Re(a_ij b_ji): 18 multiply-adds for two matrices
template <class T> __device__ __forceinline__ T v_real_trace_mul(const Mat3<T>& a, const Mat3<T>& b) {
    T s0 = 0, s1 = 0, s2 = 0;
#pragma unroll
    for (int j = 0; j < 3; j++) {
        s0 = fma(a.e[j].re, b.e[j * 3].re, s0);         s0 = fma(-a.e[j].im, b.e[j * 3].im, s0);
        s1 = fma(a.e[3 + j].re, b.e[j * 3 + 1].re, s1); s1 = fma(-a.e[3 + j].im, b.e[j * 3 + 1].im, s1);
        s2 = fma(a.e[6 + j].re, b.e[j * 3 + 2].re, s2); s2 = fma(-a.e[6 + j].im, b.e[j * 3 + 2].im, s2);
    }
    return s0 + s1 + s2;
}
template <class T> __device__ __forceinline__ T v_real_trace_mul(T s, const Mat3<T>& b) { return s * v_trace(b).re; }
template <class T> __device__ __forceinline__ T v_real_trace_mul(const Mat3<T>& a, T s) { return s * v_trace(a).re; }
template <class A, class B> struct Real<Trace<Product<A, B>>> : Node {
    template <class T> __device__ __forceinline__ static T eval(const Env<T>& e) {
        return v_real_trace_mul(A::template eval<T>(e), B::template eval<T>(e));
    }
};

template <class E> struct Norm2 : Node {
    template <class T> __device__ __forceinline__ static T eval(const Env<T>& e) { return v_norm2(E::template eval<T>(e)); }
};
template <class A, class B> struct Inner : Node {
    template <class T> __device__ __forceinline__ static Cx<T> eval(const Env<T>& e) {
        return v_inner(A::template eval<T>(e), B::template eval<T>(e));
    }
};
template <class E> struct Imag : Node {
    template <class T> __device__ __forceinline__ static T eval(const Env<T>& e) { return v_imag(E::template eval<T>(e)); }
};

// ---- the surface syntax (build-time expressions; jit.cu writes the node types out directly) -----
#ifndef __CUDACC_RTC__
template <class A, class B, class = std::enable_if_t<is_node<A> && is_node<B>>>
constexpr Product<A, B> operator*(A, B) { return {}; }
template <class A, class B, class = std::enable_if_t<is_node<A> && is_node<B>>>
constexpr Sum<A, B> operator+(A, B) { return {}; }
template <class A, class B, class = std::enable_if_t<is_node<A> && is_node<B>>>
constexpr Diff<A, B> operator-(A, B) { return {}; }
template <class E, class = std::enable_if_t<is_node<E>>> constexpr Neg<E> operator-(E) { return {}; }
template <class E> constexpr Adjoint<E> adj(E) { return {}; }
template <class E> constexpr Trace<E> trace(E) { return {}; }
template <class E> constexpr Real<E> real(E) { return {}; }
template <class E> constexpr Imag<E> imag(E) { return {}; }
template <int MU, int SIGN, class E> constexpr Shifted<E, MU, SIGN> shift(E) { return {}; }
template <class E> constexpr ShiftedRt<E> shift_rt(E) { return {}; }
#endif

// ---- kernels ---------------------------------------------------------------------------------------
template <class T> __device__ __forceinline__ void store_value(typename Vec2<T>::type* p, const Mat3<T>& v) { st_mat_at<T>(p, v); }
template <class T> __device__ __forceinline__ void store_value(typename Vec2<T>::type* p, const Spinor<T>& v) {
#pragma unroll
    for (int c = 0; c < 12; c++) {
        typename Vec2<T>::type o;
        o.x = v.e[c].re; o.y = v.e[c].im;
        p[c * kLane] = o;
    }
}
template <class T> __device__ __forceinline__ void store_value(typename Vec2<T>::type* p, const Cx<T>& v) {
    typename Vec2<T>::type o;
    o.x = v.re; o.y = v.im;
    *p = o;
}

// dst[first component cd of nd](x) = E(x) for x in the subset; other sites untouched
template <class T, class E>
__device__ __forceinline__ void assign_body(const Geom& g, const Args& a, typename Vec2<T>::type* dst, int nd, int cd, int subset) {
    const int i = blockIdx.x * 128 + threadIdx.x;
    int p, h;
    if (i >= work_items(g, subset) || !work_site(g, subset, i, p, h)) return;
    const Env<T> e{g, site_decode(g, p, h), a};
    store_value<T>(site_ptr(dst, nd, cd, e.x.index(g)), E::template eval<T>(e));
}
template <class T, class E>
__global__ void __launch_bounds__(128) assign_kernel(Geom g, Args a, typename Vec2<T>::type* dst, int nd, int cd, int subset) {
    assign_body<T, E>(g, a, dst, nd, cd, subset);
}

// result[k] = scale[k] * sum_{x in subset} Ek(x), k = 0, 1: two real-valued expressions, fp64 accumulation, fixed order.
// Persistent warps (warp w takes the 32-site items w, w + W, ...) and the warp-level deterministic tree of reduce.cuh.
template <class T, class E0, class E1>
__global__ void __launch_bounds__(128, sizeof(T) == 8 ? 2 : 4) sum2_kernel(Geom g, Args a, int subset, ReduceBuf rb, double s0, double s1) {
    const int lane = threadIdx.x & 31;
    const int nwarps = gridDim.x * 4;
    const int nitems = (work_items(g, subset) + 31) >> 5;
    double acc[2] = {0.0, 0.0};
    for (int wi = blockIdx.x * 4 + (threadIdx.x >> 5); wi < nitems; wi += nwarps) {
        const int i = wi * 32 + lane;
        int p, h;
        if (!(i < work_items(g, subset) && work_site(g, subset, i, p, h))) continue;
        const Env<T> e{g, site_decode(g, p, h), a};
        acc[0] += (double)E0::template eval<T>(e);
        acc[1] += (double)E1::template eval<T>(e);
    }
    const double sc[2] = {s0, s1};
    warp_grid_reduce<2>(acc, rb, sc);
}

// result[0, 1] = (re, im) of sum_{x in subset} E(x) for one real- or complex-valued expression, evaluated once per site
template <class T> __device__ __forceinline__ double part_re(T v) { return (double)v; }
template <class T> __device__ __forceinline__ double part_im(T) { return 0.0; }
template <class T> __device__ __forceinline__ double part_re(const Cx<T>& v) { return (double)v.re; }
template <class T> __device__ __forceinline__ double part_im(const Cx<T>& v) { return (double)v.im; }
template <class T, class E>
__device__ __forceinline__ void sumv_body(const Geom& g, const Args& a, int subset, const ReduceBuf& rb) {
    const int lane = threadIdx.x & 31;
    const int nwarps = gridDim.x * 4;
    const int nitems = (work_items(g, subset) + 31) >> 5;
    double acc[2] = {0.0, 0.0};
    for (int wi = blockIdx.x * 4 + (threadIdx.x >> 5); wi < nitems; wi += nwarps) {
        const int i = wi * 32 + lane;
        int p, h;
        if (!(i < work_items(g, subset) && work_site(g, subset, i, p, h))) continue;
        const Env<T> e{g, site_decode(g, p, h), a};
        const auto v = E::template eval<T>(e);
        acc[0] += part_re(v);
        acc[1] += part_im(v);
    }
    warp_grid_reduce<2>(acc, rb, nullptr);
}

#ifndef __CUDACC_RTC__
template <class T, class E>
cudaError_t launch_assign(const Geom& g, const Args& a, void* dst, int nd, int cd, int subset, cudaStream_t st) {
    const int items = subset == 0 ? 2 * ((g.Vh + 31) & ~31) : g.Vh;
    assign_kernel<T, E><<<(items + 127) / 128, 128, 0, st>>>(g, a, static_cast<typename Vec2<T>::type*>(dst), nd, cd, subset);
    g_launch_count++;
    return cudaGetLastError();
}
template <class T, class E0, class E1>
cudaError_t launch_sum2(const Geom& g, const Args& a, int subset, const ReduceBuf& rb, double s0, double s1, cudaStream_t st) {
    const int items = subset == 0 ? 2 * g.Vhp : g.Vh;
    int grid = (items + 127) / 128;
    const int cap = device_sm_count() * (sizeof(T) == 8 ? 2 : 4);
    if (grid > cap) grid = cap;
    sum2_kernel<T, E0, E1><<<grid, 128, 0, st>>>(g, a, subset, rb, s0, s1);
    g_launch_count++;
    return cudaGetLastError();
}

#endif   // !__CUDACC_RTC__

}  // namespace ex
}  // namespace qdp
