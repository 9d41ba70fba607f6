/*
 * qdp_b200.h -- C ABI of libqdp_b200.so: site-parallel evaluation of QDP++-style
 * lattice-field expressions on one NVIDIA B200 (sm_100a).
 *
 * This is the hot path arXiv:1111.5596 (F. Winter, "Accelerating QDP++/Chroma on
 * GPUs", PoS Lattice 2011) moves to the GPU: "data parallel types and
 * expressions suitable for lattice field theory" (sec. 1), one
 * device kernel per expression with no lattice-sized temporaries (PAPER.md:27,
 * 88-90), for the "non-kernel routines like smearing" (sec. 3) and
 * the "residual calculation and solution reconstruction" around the solver
 * (sec. 4.3).  The paper defines none of the expressions
 * mathematically; the definitions are the textbook ones fixed by
 * BASELINE.json:north_star and written out in SURVEY.md sec. 8(c) (cited below
 * as "def. N") and DESIGN.md.  The paper's run-time code generator and software
 * LRU cache are prior art and are not part of this library: fields live in
 * device memory for their whole lifetime, in a site-fastest structure-of-arrays
 * complex layout -- the coalesced layout PAPER.md:118 (sec. 6) found 6-10x
 * faster than the host-native one.
 *
 * Conventions
 *   - Every function returns a status (QDP_OK or a negative error); no C++
 *     exception crosses the ABI.  qdp_last_error() returns a thread-local
 *     message for the last failure on the calling thread.
 *   - "host" pointers are ordinary host memory owned by the caller (pinned memory
 *     makes the copies faster, it is not required).  "device" pointers are CUDA
 *     device memory on the lattice's device.
 *   - Public site order (host buffers, exported tables):
 *         lex(x) = x0 + L0*(x1 + L1*(x2 + L2*x3)),  x = (x0,x1,x2,x3), x0 fastest.
 *     The device-internal site order is private.
 *   - Host field layout, array of structures, element type = field precision,
 *     complex = (re, im) adjacent:
 *         QDP_COLOR_MATRIX  host[(lex*3 + row)*3 + col]
 *         QDP_GAUGE         host[((lex*4 + mu)*3 + row)*3 + col]
 *         QDP_FERMION       host[(lex*4 + spin)*3 + colour]
 *         QDP_COMPLEX       host[lex]
 *     (U psi)_row = sum_col U[row][col] psi[col].
 *   - Subsets: parity(x) = (x0+x1+x2+x3) & 1; QDP_EVEN = parity 0.  An operation
 *     under a subset writes only the subset's sites of its destination (all
 *     other sites keep their previous contents) and reductions sum only the
 *     subset's sites.  Neighbours are read from wherever they are.
 *   - Kernels are enqueued on the lattice's stream (default: the legacy default
 *     stream).  Field->field calls are asynchronous with respect to the host;
 *     calls that return host scalars return only when the result is complete: the
 *     reducing kernel writes it to mapped pinned host memory followed by a
 *     completion number, which the call polls (everything enqueued on that stream
 *     before it has finished by then; qdp_sum synchronises the stream instead).
 *   - Neighbour-reading operations are out of place: passing the destination as
 *     a neighbour-read source returns QDP_ERR_ALIAS.
 *   - There is no CPU fallback anywhere: a missing device is an error.
 */
#ifndef QDP_B200_H
#define QDP_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

enum {
    QDP_OK = 0,
    QDP_ERR_ARG = -1,      /* null pointer, bad enum value, bad mu/sign            */
    QDP_ERR_DIMS = -2,     /* an extent is odd or < 2, or the volume is too large  */
    QDP_ERR_KIND = -3,     /* a field has the wrong kind for this operation        */
    QDP_ERR_PREC = -4,     /* operands of different precision                      */
    QDP_ERR_LATTICE = -5,  /* operands belong to different lattices                */
    QDP_ERR_ALIAS = -6,    /* destination aliases a neighbour-read source          */
    QDP_ERR_OOM = -7,      /* device allocation failed                             */
    QDP_ERR_CUDA = -8      /* any other CUDA runtime error (message has details)   */
};

typedef enum { QDP_ALL = 0, QDP_EVEN = 1, QDP_ODD = 2 } qdp_subset;
typedef enum { QDP_F32 = 0, QDP_F64 = 1 } qdp_prec;
typedef enum {
    QDP_COLOR_MATRIX = 0,  /* 3x3 complex per site (9 complex)          */
    QDP_GAUGE = 1,         /* 4 colour matrices per site (36 complex)   */
    QDP_FERMION = 2,       /* 4 spin x 3 colour per site (12 complex)   */
    QDP_COMPLEX = 3        /* one complex number per site: the value of trace(...) in the expression layer.
                              Supported by alloc/wrap/free/bytes/upload/download/copy, qdp_sum and as the
                              destination of qdp_expr_trace_mul; every other call returns QDP_ERR_KIND. */
} qdp_kind;

typedef struct qdp_lattice qdp_lattice;   /* opaque */
typedef struct qdp_field qdp_field;       /* opaque */

/* ---- lattice ------------------------------------------------------------- */

/* Create a periodic 4-D lattice on CUDA device `device`.
 * dims (host, 4 ints): extents (L0,L1,L2,L3) = (x,y,z,t).  Every extent must be
 * even and >= 2 (red/black colouring needs it, reading A2) and the volume must
 * be below 2^31/36 sites; otherwise QDP_ERR_DIMS.  *out is owned by the caller
 * until qdp_lattice_destroy.  Fields must be freed before their lattice. */
int qdp_lattice_create(const int dims[4], int device, qdp_lattice** out);
int qdp_lattice_destroy(qdp_lattice* lat);

/* Use `cuda_stream` (a cudaStream_t, e.g. torch.cuda.current_stream().cuda_stream;
 * NULL = legacy default stream) for every later call on this lattice. */
int qdp_lattice_set_stream(qdp_lattice* lat, void* cuda_stream);

/* Sweep order of the neighbour-reading kernels (plaquette, APE step, hop): a tuning knob, results
 * do not depend on it except for the summation order of the fused reductions.  x2_extent = 0:
 * linear order (x3 slowest over the whole lattice).  x2_extent = c > 0: slabs of c values of x2
 * (x0, x1 complete) are swept one after the other, x3 slowest inside a slab, so that the links
 * of x + 3 are still in L2 when the sweep reaches them as own links.
 * qdp_lattice_create picks the value from the lattice size (slabs of <= 16 MB per x3-slice when a
 * whole slice of an fp64 gauge field exceeds 24 MB).  Returns QDP_ERR_ARG unless c divides L2
 * and L0/2 * L1 is a multiple of 32.  The reading of subsets, sites and values is unchanged
 * (SURVEY.md 8(a) rows a1, a10). */
int qdp_lattice_set_sweep_slab(qdp_lattice* lat, int x2_extent);

/* Kernel variant of qdp_plaquette and qdp_ape_smear_step: a tuning knob, results agree to rounding.
 * on = 1: on lattices whose x0 rows tile a 32-site block (L0/2 a power of two <= 32 and
 * L0/2 * L1 a multiple of 32, e.g. 32^3 x 64) and for the ALL subset, run the warp-specialised
 * kernels that stage lattice tiles in shared memory with cp.async.bulk + mbarrier rings
 * (BASELINE.json north_star: "shared-memory halo staging of a lattice tile").
 * on = 0 (default, the faster variant as measured: DESIGN.md section 4): always run the thread-per-site kernels
 * (the only variant on other lattices and subsets). */
int qdp_lattice_set_staged(qdp_lattice* lat, int on);

/* Replace the device allocator used by qdp_field_alloc and the library's scratch
 * buffers (default cudaMalloc/cudaFree).  alloc(bytes, ctx) returns a device
 * pointer aligned to >= 256 bytes or NULL; free_(ptr, ctx) releases it.  Lets
 * PyTorch's caching allocator own the memory.  Process-wide; set it before
 * creating lattices.  Passing alloc = NULL restores the default. */
int qdp_set_allocator(void* (*alloc)(size_t bytes, void* ctx),
                      void (*free_)(void* ptr, void* ctx), void* ctx);

/* Export geometry in the PUBLIC numbering for parity checks (def. 1, App. A):
 *   out[lex(x)] = lex(x + sign*mu_hat)   (V int32, host)
 *   out[lex(x)] = parity(x)              (V bytes, host)
 * Both are produced on the device by the same index arithmetic the kernels use
 * and converted to the public numbering.  Synchronous. */
int qdp_lattice_neighbor_table(qdp_lattice* lat, int mu, int sign, int32_t* host_out);
int qdp_lattice_parity_mask(qdp_lattice* lat, uint8_t* host_out);
int qdp_lattice_volume(const qdp_lattice* lat, int64_t* out);

/* Thread safety: a lattice handle (its stream, scratch partials, result and staging buffers) and
 * the fields on it must be used by one host thread at a time; different lattices may be driven
 * from different threads concurrently.  Calls that return host scalars serialise on the lattice's
 * scratch buffers by synchronising its stream.  qdp_last_error() is thread-local;
 * qdp_kernel_launch_count() is atomic; qdp_set_allocator is process-wide (set it before threads start). */

/* ---- fields -------------------------------------------------------------- */

/* Allocate a field on the lattice's device (library-owned, contents undefined). */
int qdp_field_alloc(qdp_lattice* lat, qdp_kind kind, qdp_prec prec, qdp_field** out);
/* Wrap caller-owned device memory (e.g. a torch tensor) as a field.  `bytes` must
 * be at least qdp_field_bytes(); dev_ptr must be 256-byte aligned and must stay
 * valid until qdp_field_free, which does not free it.  qdp_field_free (of either kind of
 * field) first waits for the work enqueued on the lattice's stream, so after it returns the
 * memory may be released or reused on any stream. */
int qdp_field_wrap(qdp_lattice* lat, qdp_kind kind, qdp_prec prec, void* dev_ptr, size_t bytes,
                   qdp_field** out);
int qdp_field_free(qdp_field* f);
/* Bytes of device memory a field of this kind/precision occupies.  Equal to the host
 * buffer size V * ncomp * sizeof(complex) when V/2 is a multiple of 32 (all BASELINE
 * configs); otherwise slightly larger (padding lanes of the blocked device layout). */
int qdp_field_bytes(const qdp_lattice* lat, qdp_kind kind, qdp_prec prec, size_t* out);

/* Host (layout above) <-> device (private layout).  Synchronous: the host buffer
 * may be reused as soon as the call returns.  Bit-exact round trip. */
int qdp_field_upload(qdp_field* f, const void* host_aos_lex);
int qdp_field_download(const qdp_field* f, void* host_aos_lex);
/* dst = src on the device (same kind and precision); asynchronous. */
int qdp_field_copy(qdp_field* dst, const qdp_field* src);

/* ---- expressions --------------------------------------------------------- */

/* def. 1: dst(x) = src(x + sign*mu_hat) for x in subset, coordinates mod L.
 * mu in 0..3, sign = +1 or -1; dst and src of the same kind and precision;
 * dst == src is QDP_ERR_ALIAS.  Pure data movement: bit-exact. */
int qdp_shift(qdp_field* dst, const qdp_field* src, int mu, int sign, qdp_subset subset);

/* def. 2: with P_{mu nu}(x) = U_mu(x) U_nu(x+mu) U_mu(x+nu)^dag U_nu(x)^dag and N
 * the number of sites in the subset,
 *   out[0] = 1/(6*3*N) sum_{x in subset} sum_{mu<nu} Re tr P_{mu nu}(x)
 *   out[1] = 1/(3*3*N) ... over the 3 spatial planes (mu < nu < 3)
 *   out[2] = 1/(3*3*N) ... over the 3 temporal planes (nu = 3)
 * u: QDP_GAUGE.  out: 3 doubles on the host.  Per-site arithmetic in the field
 * precision, sums accumulated in fp64 by a fixed-shape tree (bit-identical from
 * run to run).  Synchronous. */
int qdp_plaquette(const qdp_field* u, qdp_subset subset, double out[3]);

/* def. 3-4: one APE smearing step with SU(3) reprojection.  For x in subset,
 * mu in the smeared set S ({0,1,2} if t_dir == 3, {0,1,2,3} if t_dir == -1):
 *   V = (1-alpha) U_mu(x) + (alpha/n) sum_{nu in S, nu != mu}
 *         [ U_nu(x) U_mu(x+nu) U_nu(x+mu)^dag
 *         + U_nu(x-nu)^dag U_mu(x-nu) U_nu(x-nu+mu) ],      n = 2(|S|-1)
 *   u_out_mu(x) = V (V^dag V)^{-1/2} exp(-i arg(det V)/3),   arg in (-pi, pi]
 * and u_out_3(x) = u_in_3(x) (bit-exact copy) when t_dir == 3.  V must be
 * non-singular (reading A10).  u_in, u_out: QDP_GAUGE, same precision;
 * u_out == u_in is QDP_ERR_ALIAS.  alpha is cast to the field precision.
 * Asynchronous. */
int qdp_ape_smear_step(qdp_field* u_out, const qdp_field* u_in, double alpha, int t_dir,
                       qdp_subset subset);

/* SURVEY.md 8(f) row f1, first step -- one fused binary colour-matrix expression, the building
 * block of QDP++ expressions such as  m = u[mu] * shift(adj(u[nu]), FORWARD, mu):
 *   dst[slot_d](x) = opA(a[slot_a](x)) * opB(b[slot_b](x + sign*mu)),   x in subset,
 * op = adjoint if adj_a / adj_b is non-zero, else identity.  mu = 0..3 with sign = +1 | -1
 * shifts the second operand (def. 1); mu = -1: no shift.  A slot is one 3x3 matrix of a field:
 * 0 for QDP_COLOR_MATRIX, the link index 0..3 for QDP_GAUGE (QDP_ERR_ARG otherwise; QDP_FERMION
 * fields are QDP_ERR_KIND).  dst may share a field with an operand, but if mu >= 0 the slot
 * written must not be the shifted operand's slot of the same field (QDP_ERR_ALIAS).
 * Asynchronous. */
int qdp_matmul(qdp_field* dst, int slot_d, const qdp_field* a, int slot_a, int adj_a,
               const qdp_field* b, int slot_b, int adj_b, int mu, int sign, qdp_subset subset);

/* Row f1, colour matrix times fermion:  chi(x) = opA(a[slot_a](x)) psi(x + sign*mu),  x in subset;
 * the matrix acts on the colour index of each spin component.  Slots, adj_a, mu, sign as in
 * qdp_matmul.  chi, psi: QDP_FERMION; chi == psi is allowed only without a shift (mu = -1),
 * otherwise QDP_ERR_ALIAS.  Asynchronous. */
int qdp_matvec(qdp_field* chi, const qdp_field* a, int slot_a, int adj_a, const qdp_field* psi,
               int mu, int sign, qdp_subset subset);

/* SURVEY.md 8(f) row f2 (alternative projections) -- every 3x3 matrix of the sites in the subset
 * projected to SU(3):
 *   method QDP_REUNIT_POLAR (0):        Proj of def. 4 (unitary polar factor, determinant phase
 *                                       removed; gauge covariant; what the APE step applies);
 *   method QDP_REUNIT_GRAM_SCHMIDT (1): row0 normalised, row1 orthogonalised against it and
 *                                       normalised, row2 = conj(row0 x row1) (cheaper, not covariant).
 * u_out, u_in: QDP_GAUGE or QDP_COLOR_MATRIX of the same kind and precision; site-local, so
 * u_out == u_in is allowed.  Arithmetic in fp64 for both precisions.  Asynchronous.
 * Conditioning: Proj is invariant under V -> c V (c > 0) and is evaluated on V / |V|_F, then
 * polished by Newton-Schulz steps until V^dag V = 1 to ~50 ulp; the result is accurate to about
 * cond(V) * 2^-52 per matrix for cond(V) up to ~1e5 (singular V of non-zero norm: undefined, no
 * error is raised).  Under QDP_REUNIT_POLAR a matrix that is exactly zero, or has an infinite or
 * NaN entry, has no polar factor and is copied to u_out unchanged (never turned into NaNs). */
enum { QDP_REUNIT_POLAR = 0, QDP_REUNIT_GRAM_SCHMIDT = 1 };
int qdp_reunitarize(qdp_field* u_out, const qdp_field* u_in, int method, qdp_subset subset);

/* Row f2, iterative max-Re-tr projection (Cabibbo-Marinari sweeps): every 3x3 matrix V of the subset's sites is
 * replaced by X in SU(3) obtained as follows (reading in DESIGN.md section 2, f2; the paper only names "smearing"):
 *   X_0 = Gram-Schmidt(V) (QDP_REUNIT_GRAM_SCHMIDT above); one iteration = the SU(2) subgroups acting on the index
 *   pairs (0,1), (1,2), (0,2) in that order; for the pair (i,j), with m the 2x2 block of M = X V^dag in rows and
 *   columns (i,j):  r0 = Re(m00 + m11), r1 = -Im(m01 + m10), r2 = -Re(m01 - m10), r3 = -Im(m00 - m11),
 *   a = [[r0 + i r3, r2 + i r1], [-r2 + i r1, r0 - i r3]] / |r|  (the SU(2) element maximising Re tr(a m)),
 *   X <- A X with A = a embedded in (i,j).  No update can decrease Re tr(X V^dag); an SU(3) input is a fixed point.
 * `iterations` (0..1000) sweeps are always executed (no convergence test, so the result is a function of V and the
 * count only).  Same fields / aliasing rules as qdp_reunitarize; fp64 arithmetic for both precisions.  Asynchronous. */
int qdp_project_max_retr(qdp_field* u_out, const qdp_field* u_in, int iterations, qdp_subset subset);

/* def. 5: chi(x)_{s a} = sum_mu sum_b [ U_mu(x)_{ab} psi(x+mu)_{s b}
 *                                      + conj(U_mu(x-mu)_{ba}) psi(x-mu)_{s b} ]
 * for x in subset (no gamma matrices, no kappa, periodic in all directions).
 * chi, psi: QDP_FERMION; u: QDP_GAUGE; chi == psi is QDP_ERR_ALIAS.  Asynchronous. */
int qdp_hop(qdp_field* chi, const qdp_field* u, const qdp_field* psi, qdp_subset subset);

/* def. 6: chi = a*psi + b*hop(psi) on the subset, one fused kernel.  If norm2_out
 * is not NULL it receives sum_{x in subset} |chi(x)|^2 accumulated in the same
 * pass (fp64) and the call is synchronous; otherwise asynchronous.  a, b are cast
 * to the field precision. */
int qdp_axpy_hop(qdp_field* chi, double a, double b, const qdp_field* u, const qdp_field* psi,
                 qdp_subset subset, double* norm2_out);

/* one step of gauge-covariant quark smearing (Wuppertal / Gaussian:
 * the source and sink smearing stages SRC, SNK of the paper's Fig. 4):
 *   chi(x) = a psi(x) + b sum_{mu != t_dir} [ U_mu(x) psi(x+mu) + U_mu(x-mu)^dag psi(x-mu) ]
 * for x in subset.  t_dir = 3: spatial hops only (time-slices never mix); t_dir = -1: all four
 * directions, identical to qdp_axpy_hop; anything else is QDP_ERR_ARG.  Same fields, aliasing
 * rule, norm2_out behaviour and casts as qdp_axpy_hop. */
int qdp_smear_hop(qdp_field* chi, double a, double b, const qdp_field* u, const qdp_field* psi,
                  int t_dir, qdp_subset subset, double* norm2_out);

/* def. 6: global reductions over the subset, any kind; accumulated and returned
 * in fp64 for both precisions; fixed-shape tree.  Synchronous.
 *   qdp_norm2: out[0]   = sum_x sum_c |f_c(x)|^2
 *   qdp_inner: out[0,1] = (re, im) of sum_x sum_c conj(a_c(x)) b_c(x)
 *   qdp_sum:   out[2c], out[2c+1] = (re, im) of sum_x f_c(x), c < ncomp (9/36/12) */
int qdp_norm2(const qdp_field* f, qdp_subset subset, double* out);
int qdp_inner(const qdp_field* a, const qdp_field* b, qdp_subset subset, double out[2]);
int qdp_sum(const qdp_field* f, qdp_subset subset, double* out);

/* qdp_sum for callers that cannot allocate device memory (def. 6, the same sum as qdp_sum).
 *
 * Some callers hold raw device pointers and a stream and are not allowed a cudaMalloc: a plug-in
 * inside a framework whose own allocator has claimed the whole GPU, a latency-bound loop that
 * cannot take the device-wide synchronisation cudaMalloc/cudaFree imply, or code that simply has
 * no qdp_lattice (creating one allocates scratch, staging and pinned memory).  This entry point
 * needs no handle and allocates nothing, on the device or through any library routine: its
 * per-block partial sums go to a fixed 36,864-byte __device__ array compiled into the library
 * (held by every GPU that loads it, until the process exits).
 *
 *   dims        host, the four extents (even, >= 2), as for qdp_lattice_create
 *   ncomp       complex components per site, 1 <= ncomp <= 36 (QDP_COMPLEX 1, QDP_COLOR_MATRIX 9,
 *               QDP_FERMION 12, QDP_GAUGE 36).  More than 36 does not fit the fixed scratch:
 *               QDP_ERR_ARG, message names the limit
 *   field_dev   device, on the CURRENT device, a field in the library's device layout (the memory
 *               behind qdp_field_wrap / qdp_cache_acquire), read only; bytes must equal
 *               qdp_field_bytes of that lattice, kind and precision, else QDP_ERR_ARG
 *   out_dev     device-accessible (device or mapped pinned host memory), 2 * ncomp doubles:
 *               out_dev[2c], out_dev[2c+1] = (re, im) of sum_{x in subset} f_c(x), fp64, the same
 *               fixed summation order as qdp_sum (bit-identical results); caller-owned
 *   cuda_stream a cudaStream_t (NULL = legacy default stream).  Asynchronous: synchronise that
 *               stream (or order later work on it) before reading out_dev
 *
 * All calls on a device share the one scratch array, which keeps the previous call's contents;
 * nothing in it needs clearing (each call overwrites every slot it later reads).  Calls that
 * overlap on the GPU -- different streams without ordering between them -- race on it and return
 * garbage; calls on one stream are safe.  The first call on each device also looks up the array's
 * device address (cudaGetSymbolAddress; may load the library's device code): make that first call
 * outside any stream capture.  Errors: QDP_ERR_ARG / QDP_ERR_DIMS before any launch, QDP_ERR_CUDA
 * for a failed look-up or launch; nothing is written on error. */
int qdp_sum_noalloc(const int dims[4], int ncomp, qdp_prec prec, const void* field_dev, size_t bytes,
                    qdp_subset subset, double* out_dev, void* cuda_stream);

/* dst = a*x + b*y on the subset, real a, b cast to the field precision, any kind (all three
 * fields of the same kind and precision): the residual and solution-reconstruction expressions
 * around the solver (r = b - A x, x += alpha p).  Element-wise, so dst may be x or y.
 * If norm2_out is not NULL it receives sum_{x in subset} |dst(x)|^2 accumulated in the same pass
 * (fp64) and the call is synchronous; otherwise asynchronous. */
int qdp_axpby(qdp_field* dst, double a, const qdp_field* x, double b, const qdp_field* y,
              qdp_subset subset, double* norm2_out);

/* time-slice sums, the reduction under every hadron two-point function
 * (the HAD stage of the paper's Fig. 4):
 *   out[2t], out[2t+1] = (re, im) of sum_{x in subset, x3 = t} sum_c conj(a_c(x)) b_c(x),  t < L3.
 * out: host, 2*L3 doubles.  a == b gives the per-slice norm (the pion correlator of a propagator
 * column).  Same kinds/precisions rule as qdp_inner; fp64 accumulation, fixed summation order.
 * Synchronous. */
int qdp_inner_timeslices(const qdp_field* a, const qdp_field* b, qdp_subset subset, double* out);

/* Row f3, meson contractions: the same sums with a spin matrix inserted,
 *   out[2t], out[2t+1] = sum_{x in subset, x3 = t} sum_{s' s c} conj(a_{s' c}(x)) Gamma(n)_{s' s} b_{s c}(x),
 * a, b: QDP_FERMION.  Gamma(n) = g0^n0 g1^n1 g2^n2 g3^n3, n = n0 + 2 n1 + 4 n2 + 8 n3 in 0..15 (Gamma(15) = gamma_5),
 * Euclidean Hermitian gamma matrices in the DeGrand-Rossi basis (the QDP++ convention):
 *   g0 = [[0,0,0,i],[0,0,i,0],[0,-i,0,0],[-i,0,0,0]]    g1 = [[0,0,0,-1],[0,0,1,0],[0,1,0,0],[-1,0,0,0]]
 *   g2 = [[0,0,i,0],[0,0,0,-i],[-i,0,0,0],[0,i,0,0]]    g3 = [[0,0,1,0],[0,0,0,1],[1,0,0,0],[0,1,0,0]]
 * With a, b columns of quark propagators this is the building block of meson two-point functions
 * (HAD stage).  n = 0 equals qdp_inner_timeslices.  Synchronous. */
int qdp_inner_timeslices_gamma(const qdp_field* a, const qdp_field* b, int n, qdp_subset subset, double* out);

/* Row f3, baryon contractions (HAD stage: "hadron spectrum (mesonic and baryonic)"): three quark
 * fields contracted to a colour singlet with the antisymmetric tensor, the spin matrix Gamma(n) (as in
 * qdp_inner_timeslices_gamma) between the first two, summed per time-slice; the third quark's spin index g stays open:
 *   out[t][g] = sum_{x in subset, x3 = t} sum_{(a',b',c')} eps_{a'b'c'} sum_{a b c} eps_{abc}
 *               [ sum_{al be} q1[a']_{al a}(x) Gamma(n)_{al be} q2[b']_{be b}(x) ] q3[c']_{g c}(x).
 * nsrc = 3: q1, q2, q3 point to three QDP_FERMION fields each, one per SOURCE colour a', b', c' (columns of a quark
 * propagator with fixed source spin), and (a',b',c') runs over the six permutations with their signs: the
 * eps_{abc} eps_{a'b'c'} colour contraction of a nucleon-type two-point function, all nine fields read in one pass.
 * nsrc = 1: one field per quark and no source contraction (the colour-singlet operator of three spinor fields).
 * No complex conjugation is applied to any field.  out: host, 8*L3 doubles, out[(t*4 + g)*2 + (0: re, 1: im)].
 * fp64 accumulation, fixed summation order.  All fields on one lattice and of one precision.  Synchronous. */
int qdp_baryon_timeslices(const qdp_field* const* q1, const qdp_field* const* q2, const qdp_field* const* q3,
                          int nsrc, int n, qdp_subset subset, double* out);

/* ---- the expression layer ---------------------------------------------
 * The paper turns every QDP++ expression (PETE expression templates, "expressions that look like their
 * mathematical counterparts") into one generated kernel.  Here the
 * expression is a C++ type built with *, +, adj, trace, real, shift (csrc/expr.cuh) and nvcc
 * instantiates ONE kernel per expression at build time, with an optional fused global sum; no
 * temporaries, no JIT.  The calls below are named instantiations; their definitions are the same as
 * those of the hand-fused calls above (def. 2, def. 3 of SURVEY.md 8(c)).
 *
 *   qdp_expr_plaquette:  sum_x real(trace(u[mu] * shift(u[nu],+mu) * adj(shift(u[mu],+nu)) * adj(u[nu]))) summed over
 *                        the six planes in one kernel; out[3] normalised exactly as qdp_plaquette.  Synchronous.
 *   qdp_expr_staple:     dst(x) = sum_{nu != mu, nu != t_dir} [ u[nu] * shift(u[mu],+nu) * adj(shift(u[nu],+mu))
 *                                 + shift(adj(u[nu]) * u[mu] * shift(u[nu],+mu), -nu) ](x), x in subset: the staple sum
 *                        S_mu of def. 3 (t_dir = 3: spatial, 4 staples; -1: all directions, 6).  dst: QDP_COLOR_MATRIX,
 *                        u: QDP_GAUGE, same lattice and precision; mu must be a smeared direction.  Asynchronous.
 *   qdp_expr_ape_blend:  dst = (1-alpha) * u[mu] + (alpha/n) * S_mu, n = 4 or 6: the APE link before projection
 *                        (qdp_reunitarize(dst, dst, QDP_REUNIT_POLAR) then gives the link of qdp_ape_smear_step).
 *   qdp_expr_trace_mul:  dst(x) = trace(opA(a[slot_a])(x) * opB(b[slot_b])(x + sign*mu)), dst: QDP_COMPLEX; slots, op and
 *                        mu = -1 (no shift) as in qdp_matmul.  Asynchronous.
 *   qdp_expr_sum_trace_mul: out = (re, im) of sum_{x in subset} of that trace (fp64 accumulation, fixed order); with
 *                        a = u', b = u, adj_b = 1 it is the link overlap sum tr(U' U^dag) used to monitor smearing.
 *                        Synchronous. */
int qdp_expr_plaquette(const qdp_field* u, qdp_subset subset, double out[3]);
int qdp_expr_staple(qdp_field* dst, const qdp_field* u, int mu, int t_dir, qdp_subset subset);
int qdp_expr_ape_blend(qdp_field* dst, const qdp_field* u, int mu, double alpha, int t_dir, qdp_subset subset);
int qdp_expr_trace_mul(qdp_field* dst, const qdp_field* a, int slot_a, int adj_a, const qdp_field* b, int slot_b,
                       int adj_b, int mu, int sign, qdp_subset subset);
int qdp_expr_sum_trace_mul(const qdp_field* a, int slot_a, int adj_a, const qdp_field* b, int slot_b, int adj_b,
                           int mu, int sign, qdp_subset subset, double out[2]);

/* ---- Row f1, second step: run-time expressions -------------------------------------------------------------------
 * The paper's scheme itself (the tree parser "generates the CUDA kernel code" of an expression, which is
 * JIT-compiled and cached so that "each expression is compiled only once"): the expression arrives as text, is parsed
 * and type-checked on the host, written out as a node type of the expression layer (csrc/expr.cuh), compiled with NVRTC
 * for sm_100a into ONE kernel and cached by (expression, precision, assignment | sum).  The first use of an expression
 * costs one compilation (0.2-0.4 s); later uses launch the cached kernel.  libnvrtc is loaded at the first compilation
 * (QDP_ERR_CUDA with a message if it is missing); nothing is read from the file system.
 *   expr   := term { ('+' | '-') term }    term := factor { '*' factor }
 *   factor := '-' factor | adj(expr) | trace(expr) | real(expr) | imag(expr) | norm2(expr) | inner(expr, expr)
 *           | shift(expr, +mu | -mu) | '(' expr ')' | leaf
 *   leaf   := f<k> [ '[' slot ']' ]        field argument k = 0..3: matrix `slot` of a QDP_COLOR_MATRIX or QDP_GAUGE field
 *                                          (a link of a gauge field; default 0), or the spinor of a QDP_FERMION field
 *           | s<k>                         real scalar argument k = 0..3 (cast to the field precision)
 *           | number                       decimal literal (2, 0.5, 1.5e-3): a real constant; unlike a scalar argument it
 *                                          is part of the compiled expression, so another value is another kernel
 * Semantics as in the build-time layer and SURVEY.md 8(c): a value is a 3x3 matrix, a spinor (4 spin x 3 colour), a
 * complex number or a real number; adj = conjugate transpose (conjugate of a complex number; not defined on spinors),
 * trace: matrix -> complex, real / imag: complex -> real, norm2: spinor -> real (sum over spin and colour of |.|^2),
 * inner(a, b): two spinors -> complex (sum of conj(a) b), shift(e, +mu)(x) = e(x + mu) for the whole sub-expression e
 * (A3), '+' and '-' need equal kinds (a - b is the elementwise difference: the residual r = b - A x of PAPER.md:96 is
 * "f1 - s0 * (...)"), a leading '-' negates a value of any kind and binds tighter than '*', '*' is matrix * matrix, matrix * spinor (the matrix acts on the colour index of every spin
 * component: the product of the hopping term, A11), real * anything, anything * real, complex * complex or complex *
 * spinor.  All field arguments belong to one lattice and precision.  Example, the hopping term of def. 5:
 *   "f0[0] * shift(f1, +0) + shift(adj(f0[0]) * f1, -0) + f0[1] * shift(f1, +1) + ..."  with f0 = u, f1 = psi.
 *   qdp_expr_jit_kind:    host only; *kind_out = 0 matrix, 1 complex, 2 real, 3 spinor.  field_kinds[k] = qdp_kind of argument k.
 *   qdp_expr_jit_compile: host only (NVRTC needs no device): compiles the kernel for (expr, prec, sum != 0) into the
 *                         cache if it is not there; *cubin_bytes (optional) receives the size of its image.
 *   qdp_expr_jit_assign:  dst[slot_d](x) = expr(x) for x in subset, other sites untouched.  A matrix expression needs a
 *                         QDP_COLOR_MATRIX (slot_d = 0) or QDP_GAUGE destination, a spinor expression a QDP_FERMION and a
 *                         complex one a QDP_COMPLEX destination (QDP_ERR_KIND).  dst may be an operand unless the expression contains a shift (QDP_ERR_ALIAS).
 *                         Asynchronous.
 *   qdp_expr_jit_sum:     out = (re, im) of sum_{x in subset} expr(x) for a real or complex expression (fp64
 *                         accumulation, fixed order, not normalised).  Synchronous.
 *   qdp_expr_jit_compilations: number of NVRTC compilations this process has done (cache misses).
 * Syntax and kind errors are QDP_ERR_ARG with the position in qdp_last_error(). */
int qdp_expr_jit_kind(const char* expr, const int* field_kinds, int nfields, int nscalars, int* kind_out);
int qdp_expr_jit_compile(const char* expr, const int* field_kinds, int nfields, int nscalars, qdp_prec prec, int sum,
                         size_t* cubin_bytes);
int qdp_expr_jit_assign(qdp_field* dst, int slot_d, const char* expr, const qdp_field* const* fields, int nfields,
                        const double* scalars, int nscalars, qdp_subset subset);
int qdp_expr_jit_sum(const char* expr, const qdp_field* const* fields, int nfields, const double* scalars, int nscalars,
                     qdp_subset subset, double out[2]);
int64_t qdp_expr_jit_compilations(void);

/* ---- faces for an x3-slab decomposition over several GPUs ----------------------
 * The paper is single-GPU (multi-GPU "future work") and BASELINE.json fixes one GPU, so bench.py runs
 * replicas only; these calls are the device half of the decomposition SURVEY.md 8(e) describes: every rank owns a slab
 * of L3/N time-slices as a lattice of its own, a shift along x3 becomes one exchange of a boundary time-slice and a
 * global sum becomes an all-reduce of doubles (paper_1111_5596_b200/slab.py does the exchange with torch.distributed).
 *   qdp_field_get_timeslice: dev_buf <- the sites with x3 = t of f (both parities), qdp_field_timeslice_bytes(f) bytes
 *                            of device memory in a private layout that qdp_field_set_timeslice of any lattice with
 *                            the same L0, L1, L2 and a field of the same kind and precision understands.
 *   qdp_field_set_timeslice: the sites with x3 = t of f that belong to `subset` <- dev_buf; other sites untouched.
 * Both asynchronous on the lattice's stream. */
int qdp_field_timeslice_bytes(const qdp_field* f, size_t* out);
int qdp_field_get_timeslice(const qdp_field* f, int t, void* dev_buf, size_t bytes);
int qdp_field_set_timeslice(qdp_field* f, int t, const void* dev_buf, size_t bytes, qdp_subset subset);

/* ---- device memory pool and LRU residency manager --------------------------
 * The paper's memory layer: "the pool manager grabs a large chunk of GPU memory at start-up" and a
 * software cache "decides host/device affiliation per lattice object and spills least-recently-used objects" when an
 * allocation does not fit; QUDA's allocations are redirected into the same pool.  On a 180 GB B200 the
 * BASELINE workloads are resident for their lifetime, so the hot path never needs it; it is provided for working sets
 * beyond device memory.  Host-side logic (csrc/pool.cu); the policy is stated here and modelled in oracle/pool_model.py.
 *
 * Pool: one cudaMalloc of `bytes` on `device` at creation, sub-allocated in units of 256 bytes: first fit = the free
 * block with the lowest offset that is large enough; freed blocks are merged with free neighbours.  device = -1 creates
 * an address-range-only pool (nothing is allocated or copied; returned pointers are offsets from a fake base): the
 * allocator and the eviction policy can then be exercised without a GPU.  qdp_pool_alloc returns QDP_ERR_OOM only when
 * no block fits after every unlocked cached object has been spilled.  qdp_pool_stats: out = {capacity, bytes in use,
 * largest free block, number of free blocks}.  qdp_pool_hook_alloc/free have the signature qdp_set_allocator expects
 * (ctx = the pool), so fields and scratch buffers can be drawn from the pool.
 *
 * Cached objects: qdp_cache_register ties `bytes` of data to a caller-owned host buffer (pinned memory makes the
 * copies fast; it must stay valid until qdp_cache_unregister).  The data are whatever bytes the caller keeps there --
 * for a field, its device layout (qdp_field_wrap the pointer qdp_cache_acquire returns, with qdp_field_bytes bytes).
 * qdp_cache_acquire(c, for_write, &ptr): if c is not resident, allocate it from the pool -- when nothing fits, spill
 * resident objects with no outstanding acquire, least recently acquired first, one at a time until a block fits (an
 * object acquired for writing since it was paged in is first copied back to its host buffer) -- and copy the host
 * buffer in; then lock it, mark it most recently used and return its device address.  qdp_cache_release unlocks.
 * The copies are synchronous cudaMemcpy calls: work that still uses an object must have been synchronised
 * (qdp_lattice_sync) before the object is released.  qdp_cache_unregister copies a modified resident object back and
 * frees it.  qdp_pool_eviction_log lists the ids (qdp_cache_id: registration order, from 0) of the objects spilled so
 * far, oldest first; *n receives their number.  Not thread-safe: one host thread per pool. */
typedef struct qdp_pool qdp_pool;       /* opaque */
typedef struct qdp_cached qdp_cached;   /* opaque */
int qdp_pool_create(int device, size_t bytes, qdp_pool** out);
int qdp_pool_destroy(qdp_pool* pool);
int qdp_pool_alloc(qdp_pool* pool, size_t bytes, void** out);
int qdp_pool_free(qdp_pool* pool, void* ptr);
int qdp_pool_stats(const qdp_pool* pool, size_t out[4]);
void* qdp_pool_hook_alloc(size_t bytes, void* pool);
void qdp_pool_hook_free(void* ptr, void* pool);
int qdp_cache_register(qdp_pool* pool, void* host_buf, size_t bytes, qdp_cached** out);
int qdp_cache_acquire(qdp_cached* c, int for_write, void** dev_ptr);
int qdp_cache_release(qdp_cached* c);
int qdp_cache_unregister(qdp_cached* c);
int qdp_cache_is_resident(const qdp_cached* c);
int64_t qdp_cache_id(const qdp_cached* c);
int qdp_pool_eviction_log(const qdp_pool* pool, int64_t* ids, int max, int* n);

/* Block the host until every call enqueued on the lattice's stream has finished. */
int qdp_lattice_sync(qdp_lattice* lat);

/* Number of kernels this library has launched in this process (all lattices). */
int64_t qdp_kernel_launch_count(void);

const char* qdp_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* QDP_B200_H */
