// expr.cu -- named instantiations of the expression layer (expr.cuh), one kernel each:
//   qdp_expr_plaquette      sum(real(trace(u[mu] * shift(u[nu],mu) * adj(shift(u[mu],nu)) * adj(u[nu])))) over the planes
//   qdp_expr_staple         dst = sum_nu [ u[nu] * shift(u[mu],nu) * adj(shift(u[nu],mu))
//                                        + shift(adj(u[nu]) * u[mu] * shift(u[nu],mu), -nu) ]             (def. 3)
//   qdp_expr_ape_blend      dst = (1-alpha) * u[mu] + (alpha/n) * (that staple sum)
//   qdp_expr_trace_mul      dst = trace(opA(a[ia]) * opB(shift(b[ib], sign*mu)))          (complex field)
//   qdp_expr_sum_trace_mul  sum(trace(opA(a[ia]) * opB(shift(b[ib], sign*mu))))           (complex number)
// The hand-fused kernels (plaquette.cu, ape.cu) evaluate the same definitions; tests compare both with the oracle and
// bench.py reports the time of the expression form next to the hand-fused one.
#include "expr.cuh"

namespace qdp {
using namespace ex;

// ---- plaquette -------------------------------------------------------------------------------------
template <int MU, int NU>
using PlaqPlane = decltype(real(trace(U<MU>() * shift<MU, +1>(U<NU>()) * adj(shift<NU, +1>(U<MU>())) * adj(U<NU>()))));
using PlaqSpatial = decltype(PlaqPlane<0, 1>() + PlaqPlane<0, 2>() + PlaqPlane<1, 2>());
using PlaqTemporal = decltype(PlaqPlane<0, 3>() + PlaqPlane<1, 3>() + PlaqPlane<2, 3>());

// result[0] = spatial planes / (9 N), result[1] = temporal planes / (9 N); the caller averages them for all six
cudaError_t launch_expr_plaquette(int prec, const Geom& g, const void* u, int subset, const ReduceBuf& rb, cudaStream_t st) {
    Args a = {};
    a.f[0] = u; a.ncomp[0] = 36;
    const double s = 1.0 / (9.0 * (double)(subset == 0 ? g.V : g.Vh));
    return prec ? launch_sum2<double, PlaqSpatial, PlaqTemporal>(g, a, subset, rb, s, s, st)
                : launch_sum2<float, PlaqSpatial, PlaqTemporal>(g, a, subset, rb, s, s, st);
}

// ---- staple sum and APE blend (def. 3) -----------------------------------------------------------
template <int MU, int NU> using Upper = decltype(U<NU>() * shift<NU, +1>(U<MU>()) * adj(shift<MU, +1>(U<NU>())));
template <int MU, int NU> using Lower = decltype(shift<NU, -1>(adj(U<NU>()) * U<MU>() * shift<MU, +1>(U<NU>())));
template <int MU, int NU> using Staples = decltype(Upper<MU, NU>() + Lower<MU, NU>());
template <int MU, bool FOURD> struct StapleSum;
template <int MU> struct StapleSum<MU, false> {    // nu over the two other spatial directions
    using type = decltype(Staples<MU, (MU + 1) % 3>() + Staples<MU, (MU + 2) % 3>());
};
template <int MU> struct StapleSum<MU, true> {     // nu over the three other directions
    using type = decltype(Staples<MU, (MU + 1) % 4>() + Staples<MU, (MU + 2) % 4>() + Staples<MU, (MU + 3) % 4>());
};
template <int MU, bool FOURD> using Blend = decltype(Sc<0>() * U<MU>() + Sc<1>() * typename StapleSum<MU, FOURD>::type());

template <class T, int MU, bool FOURD>
static cudaError_t staple_dispatch(const Geom& g, const Args& a, void* dst, bool blend, int subset, cudaStream_t st) {
    return blend ? launch_assign<T, Blend<MU, FOURD>>(g, a, dst, 9, 0, subset, st)
                 : launch_assign<T, typename StapleSum<MU, FOURD>::type>(g, a, dst, 9, 0, subset, st);
}
template <class T>
static cudaError_t staple_dispatch_mu(const Geom& g, const Args& a, void* dst, int mu, bool fourd, bool blend, int subset,
                                      cudaStream_t st) {
    if (fourd) {
        switch (mu) {
            case 0: return staple_dispatch<T, 0, true>(g, a, dst, blend, subset, st);
            case 1: return staple_dispatch<T, 1, true>(g, a, dst, blend, subset, st);
            case 2: return staple_dispatch<T, 2, true>(g, a, dst, blend, subset, st);
            default: return staple_dispatch<T, 3, true>(g, a, dst, blend, subset, st);
        }
    }
    switch (mu) {
        case 0: return staple_dispatch<T, 0, false>(g, a, dst, blend, subset, st);
        case 1: return staple_dispatch<T, 1, false>(g, a, dst, blend, subset, st);
        default: return staple_dispatch<T, 2, false>(g, a, dst, blend, subset, st);
    }
}
// dst: colour-matrix field.  blend: dst = (1-alpha) u[mu] + (alpha/n) staples, n = 4 (t_dir = 3) or 6 (t_dir = -1)
cudaError_t launch_expr_staple(int prec, const Geom& g, void* dst, const void* u, int mu, int t_dir, bool blend, double alpha,
                               int subset, cudaStream_t st) {
    Args a = {};
    a.f[0] = u; a.ncomp[0] = 36;
    const bool fourd = t_dir < 0;
    a.sc[0] = 1.0 - alpha;
    a.sc[1] = alpha / (fourd ? 6.0 : 4.0);
    return prec ? staple_dispatch_mu<double>(g, a, dst, mu, fourd, blend, subset, st)
                : staple_dispatch_mu<float>(g, a, dst, mu, fourd, blend, subset, st);
}

// ---- trace of a binary product with run-time slots and shift ---------------------------------------
template <bool ADJ, class E> struct MaybeAdj { using type = E; };
template <class E> struct MaybeAdj<true, E> { using type = Adjoint<E>; };
template <bool ADJ_A, bool ADJ_B>
using TraceMul = Trace<Product<typename MaybeAdj<ADJ_A, Mrt<0>>::type, typename MaybeAdj<ADJ_B, ShiftedRt<Mrt<1>>>::type>>;

template <class T, bool ADJ_A, bool ADJ_B>
static cudaError_t trace_mul_go(const Geom& g, const Args& a, void* dst, int subset, const ReduceBuf& rb, cudaStream_t st) {
    using E = TraceMul<ADJ_A, ADJ_B>;
    if (dst) return launch_assign<T, E>(g, a, dst, 1, 0, subset, st);
    return launch_sum2<T, Real<E>, Imag<E>>(g, a, subset, rb, 1.0, 1.0, st);
}
// dst != nullptr: complex field dst(x) = trace(...); dst == nullptr: (re, im) of the sum over the subset through rb
cudaError_t launch_expr_trace_mul(int prec, const Geom& g, void* dst, const void* A, int na, int ia, bool adj_a, const void* B,
                                  int nb, int ib, bool adj_b, int mu, int sign, int subset, const ReduceBuf& rb, cudaStream_t st) {
    Args a = {};
    a.f[0] = A; a.ncomp[0] = na; a.slot[0] = ia;
    a.f[1] = B; a.ncomp[1] = nb; a.slot[1] = ib;
    a.mu = mu; a.sign = sign;
    if (prec) {
        if (adj_a) return adj_b ? trace_mul_go<double, true, true>(g, a, dst, subset, rb, st) : trace_mul_go<double, true, false>(g, a, dst, subset, rb, st);
        return adj_b ? trace_mul_go<double, false, true>(g, a, dst, subset, rb, st) : trace_mul_go<double, false, false>(g, a, dst, subset, rb, st);
    }
    if (adj_a) return adj_b ? trace_mul_go<float, true, true>(g, a, dst, subset, rb, st) : trace_mul_go<float, true, false>(g, a, dst, subset, rb, st);
    return adj_b ? trace_mul_go<float, false, true>(g, a, dst, subset, rb, st) : trace_mul_go<float, false, false>(g, a, dst, subset, rb, st);
}

}  // namespace qdp
