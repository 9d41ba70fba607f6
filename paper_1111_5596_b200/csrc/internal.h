// internal.h -- declarations shared by api.cu and the kernel translation units.
#pragma once
#include <atomic>
#include <cstddef>
#include <cstdint>
#include <cstring>
#include <string>
#include <cuda_runtime.h>

#include "geom.cuh"
#include "reduce.cuh"

namespace qdp {

extern std::atomic<long long> g_launch_count;   // kernels launched by this library (lattices may be driven from several host threads)
// multiprocessors of the current device (cached per device)
int device_sm_count();

// All launchers enqueue on `st` and return cudaGetLastError().
// prec: 0 = fp32, 1 = fp64 (qdp_prec).  subset: 0 all, 1 even, 2 odd.

// layout.cu
cudaError_t launch_aos_to_soa(int prec, const Geom& g, int ncomp, const void* stage, void* field,
                              int lex_begin, int nsites, cudaStream_t st);
cudaError_t launch_soa_to_aos(int prec, const Geom& g, int ncomp, const void* field, void* stage,
                              int lex_begin, int nsites, cudaStream_t st);
cudaError_t launch_neighbor_table(const Geom& g, int mu, int sign, int32_t* out_lex, cudaStream_t st);
cudaError_t launch_parity_mask(const Geom& g, uint8_t* out_lex, cudaStream_t st);

// face of the sites with x3 = t: field -> buf (to_face) or buf -> field on the sites of `subset`; buf holds 2 * ncomp * s3 elements
cudaError_t launch_timeslice(int prec, const Geom& g, int ncomp, void* field, void* buf, int t, int subset, bool to_face,
                             cudaStream_t st);

// shift.cu
cudaError_t launch_shift(int prec, const Geom& g, int ncomp, void* dst, const void* src, int mu,
                         int sign, int subset, cudaStream_t st);

// reduce.cu
cudaError_t launch_norm2(int prec, const Geom& g, int ncomp, const void* f, int subset,
                         const ReduceBuf& rb, cudaStream_t st);
cudaError_t launch_inner(int prec, const Geom& g, int ncomp, const void* a, const void* b, int subset,
                         const ReduceBuf& rb, cudaStream_t st);
// out_dev: 2*ncomp doubles on the device; partials: scratch of 2*ncomp*nblk doubles
cudaError_t launch_sum(int prec, const Geom& g, int ncomp, const void* f, int subset,
                       double* partials, double* out_dev, cudaStream_t st);

// dst = a x + b y on the subset (dst may be x or y); want_norm2: norm2(dst) through rb
cudaError_t launch_axpby(int prec, const Geom& g, int ncomp, void* dst, const void* x, const void* y, double a,
                         double b, int subset, bool want_norm2, const ReduceBuf& rb, cudaStream_t st);
// A spin matrix that is a phased permutation: (Gamma psi)_s = i^ph[s] psi_perm[s] (every product of gamma matrices is one)
struct SpinMatrix { int perm[4]; int ph[4]; };
// partials: scratch of 2*16*L3 doubles; out_dev: 2*L3 doubles on the device; gamma != nullptr (fermions only):
// a is paired with Gamma b
cudaError_t launch_inner_timeslices(int prec, const Geom& g, int ncomp, const void* a, const void* b, int subset,
                                    double* partials, double* out_dev, cudaStream_t st, const SpinMatrix* gamma = nullptr);

// hop.cu
// ndir = 4: all directions; 3: mu = 0, 1, 2 only (qdp_smear_hop with t_dir = 3)
cudaError_t launch_hop(int prec, const Geom& g, void* chi, const void* u, const void* psi, int subset,
                       bool axpy, double a, double b, bool want_norm2, const ReduceBuf& rb,
                       cudaStream_t st, int ndir = 4);

// plaquette.cu (thread per site) and plaquette_tma.cu (shared-memory staged; ALL subset, lattices whose x0 rows tile a block)
cudaError_t launch_plaquette(int prec, const Geom& g, const void* u, int subset, const ReduceBuf& rb,
                             cudaStream_t st);
bool plaquette_tma_applicable(const Geom& g, int subset);
cudaError_t launch_plaquette_tma(int prec, const Geom& g, const void* u, const ReduceBuf& rb, int sms, cudaStream_t st);

// matmul.cu: dst slot id = op(a slot ia)(x) * op(b slot ib)(x + sign*mu); mu < 0: no shift; n* = components per site
cudaError_t launch_matmul(int prec, const Geom& g, void* dst, int nd, int id, const void* a, int na, int ia, bool adj_a,
                          const void* b, int nb, int ib, bool adj_b, int mu, int sign, int subset, cudaStream_t st);

// chi(x) = op(a slot ia)(x) psi(x + sign*mu); mu < 0: no shift
cudaError_t launch_matvec(int prec, const Geom& g, void* chi, const void* a, int na, int ia, bool adj_a, const void* psi,
                          int mu, int sign, int subset, cudaStream_t st);

// reunit.cu: method 0 = Proj (polar factor, determinant phase removed), 1 = Gram-Schmidt, 2 = `iters` max-Re-tr sweeps
// from the Gram-Schmidt start; in place allowed
cudaError_t launch_reunit(int prec, const Geom& g, int ncomp, void* out, const void* in, int method, int subset,
                          cudaStream_t st, int iters = 0);

// baryon.cu: q[quark][source colour] (nsrc = 1 or 3 fields per quark); partials 8 * 16 * L3 doubles, out_dev 8 * L3
cudaError_t launch_baryon_timeslices(int prec, const Geom& g, const void* const q[3][3], int nsrc, const SpinMatrix& gm,
                                     int subset, double* partials, double* out_dev, cudaStream_t st);

// expr.cu: named instantiations of the compile-time expression layer (expr.cuh)
cudaError_t launch_expr_plaquette(int prec, const Geom& g, const void* u, int subset, const ReduceBuf& rb, cudaStream_t st);
cudaError_t launch_expr_staple(int prec, const Geom& g, void* dst, const void* u, int mu, int t_dir, bool blend, double alpha,
                               int subset, cudaStream_t st);
cudaError_t launch_expr_trace_mul(int prec, const Geom& g, void* dst, const void* A, int na, int ia, bool adj_a, const void* B,
                                  int nb, int ib, bool adj_b, int mu, int sign, int subset, const ReduceBuf& rb, cudaStream_t st);

// jit.cu: run-time expressions (text -> node type of expr.cuh -> NVRTC -> cached kernel)
enum { JIT_MAT = 0, JIT_CPLX = 1, JIT_REAL = 2, JIT_SPINOR = 3 };   // value kind of an expression: 3x3 matrix, complex, real, spin-colour vector
struct JitExpr {
    std::string type;       // the expression as a node type of expr.cuh
    int kind;
    bool has_shift;         // some operand is read at a neighbour site
    unsigned fields_used;   // bit k: field argument k occurs
};
namespace ex { struct Args; }
// ncomp[k]: components per site of field argument k (9, 36 or 12).  Returns 0, or -1 with *err set.  No device needed.
int jit_parse(const char* text, const int* ncomp, int nfields, int nscalars, JitExpr* out, std::string* err);
std::string jit_source(const JitExpr& e, int prec, bool sum);
int jit_compile_only(const JitExpr& e, int prec, bool sum, size_t* cubin_bytes, std::string* err);
long long jit_compilations();
// a failed compilation returns cudaErrorUnknown with *err set
cudaError_t jit_launch_assign(const JitExpr& e, int prec, const Geom& g, const ex::Args& a, void* dst, int nd, int cd, int subset,
                              cudaStream_t st, std::string* err);
cudaError_t jit_launch_sum(const JitExpr& e, int prec, const Geom& g, const ex::Args& a, int subset, const ReduceBuf& rb,
                           cudaStream_t st, std::string* err);

// ape.cu
cudaError_t launch_ape(int prec, const Geom& g, void* u_out, const void* u_in, double alpha, int t_dir,
                       int subset, cudaStream_t st);

}  // namespace qdp
