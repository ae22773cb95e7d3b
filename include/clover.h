/*
 * include/clover.h -- C-ABI of the B200-native Wilson-clover solve path of arXiv:1405.4524.
 *
 * What the calls compute (citations: P:L<n> = PAPER.md line n; S = SURVEY.md; R<n> = reading n in DESIGN.md):
 *   The paper's stochastic propagators need, for every random source eta_r, the solution vector
 *   X_r of  D X_r = eta_r  ("X is the solution vector and eta is the random source vector", P:L303,
 *   eq. 7.3 at P:L300), D being "the lattice fermion matrix computed in the background of the gauge
 *   fields" for "clover fermions with tree-level improved clover coefficient"; the paper
 *   hands this to a GPU inverter through an interface that "just involved some reordering of the arrays"
 *   (P:L318).  This library is that inverter and that interface.  The operator is
 *       D = A - kappa H,
 *       (H psi)(x) = sum_mu [ f_mu(x) (1 - gamma_mu) U_mu(x) psi(x+mu) + g_mu(x) (1 + gamma_mu) U_mu(x-mu)^+ psi(x-mu) ],
 *       A(x) = 1 + i c_sw kappa sum_{mu<nu} sigma_{mu nu} (x) Fhat_{mu nu}(x),
 *   with the gamma basis, boundary phases f, g and the four-leaf clover Fhat of S 8(c) O1-O4 (R1-R5).
 *
 * Canonical (ABI) layouts.  All arrays are C-ordered, complex numbers are (re, im) pairs:
 *   links    double [4 mu][T][Z][Y][X][3 row][3 col][2]     U_mu(x) stored at x, pointing x -> x+mu
 *   spinors  real   [n_rhs][T][Z][Y][X][4 spin][3 colour][2]   real = double, or float where a
 *                                                               `precision` argument says 32
 *   mu = 0,1,2,3 = x,y,z,t; dims = {X,Y,Z,T}, every extent even and >= 2; bc[mu] = +1 | -1.
 *
 * Pointers: every pointer named *_dev is a DEVICE pointer owned by the caller (e.g. torch tensor
 * data_ptr()); *_host is HOST memory (pinned for full copy speed).  `stream` is a cudaStream_t cast
 * to void* (NULL = legacy default stream).  The library never frees or keeps caller buffers: a
 * context copies what it needs during clover_create.  Workspaces are owned by the context.
 *
 * Errors: every call returns 0 on success or a negative CLOVER_E* code (no exceptions, no abort, no
 * printing).  clover_solve* additionally returns the positive count of right-hand sides that did
 * not converge.  clover_last_error() gives a message for the last failure on the calling thread.
 * There is no CPU fallback anywhere: without a CUDA device every call fails with CLOVER_ECUDA.
 */
#ifndef CLOVER_B200_H
#define CLOVER_B200_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define CLOVER_OK 0
#define CLOVER_EINVAL (-1) /* bad dims / odd extent / n_rhs out of range / null pointer / bad enum */
#define CLOVER_ECUDA (-2)  /* a CUDA runtime call failed (message has the CUDA error string)        */
#define CLOVER_ENOMEM (-3) /* device allocation failed                                              */

typedef struct clover_ctx clover_ctx; /* opaque: reordered links, A, A^-1 (fp64 + fp32), workspaces */

typedef struct {
    int recon;   /* gauge storage of the fp32 (sloppy) links: 18 = full, 12 = two rows (third row rebuilt in-kernel).
                    fp64 links are always stored in full. */
    int max_rhs; /* largest batch any later call uses (1..8); sizes the workspaces */
} clover_opts;

typedef struct {
    int status;           /* 0 converged, 1 max_iter reached, 2 repeated breakdown (still breaking down after 100 restarts of the recurrence), 3 non-finite */
    int iters;            /* BiCGStab iterations of the BATCH this source was in (the rhs of a batch iterate together; a rhs that
                             converges early is frozen, so every rhs of a batch reports the same count) */
    int reliable_updates; /* fp64 residual recomputations of that batch */
    double iter_resid;    /* the fp64 residual the convergence decision was taken on: ||b_e - Mhat y|| / ||eta|| of the last reliable
                             update, or the full-lattice residual when the final verification confirmed the claim itself */
    double true_resid;    /* full-lattice fp64 ||eta - D psi|| / ||eta||, recomputed from the returned psi */
} clover_rhs_info;

/* operators of dslash_apply (S 8(a) H3, H4; S 8(b)) */
enum {
    CLOVER_OP_HOP_EO = 0,     /* out_even = H in_odd,  out_odd = 0 */
    CLOVER_OP_HOP_OE = 1,     /* out_odd  = H in_even, out_even = 0 */
    CLOVER_OP_HOP_FULL = 2,   /* out = H in */
    CLOVER_OP_CLOVER = 3,     /* out = A in */
    CLOVER_OP_CLOVER_INV = 4, /* out = A^-1 in */
    CLOVER_OP_D_FULL = 5,     /* out = (A - kappa H) in */
    CLOVER_OP_MHAT = 6        /* out_even = (A_ee - kappa^2 H_eo A_oo^-1 H_oe) in_even, out_odd = 0 (R13) */
};

/* Build a context: reorder the links into the even-odd site-blocked layout (fp64 and fp32 copies,
 * fp32 optionally two-row compressed), build the clover term A(x) from the four-leaf Fhat (S 8(c) O3),
 * pack it as two 6x6 Hermitian blocks per site, invert the blocks (S 8(a) S0, S1).
 * gauge_dev: canonical links (device).  Synchronises `stream` before returning. */
int clover_create(clover_ctx **out, const double *gauge_dev, const int dims[4], double kappa, double c_sw,
                  const int bc[4], const clover_opts *opts, void *stream);
void clover_destroy(clover_ctx *ctx);

/* out = op(in) for n_rhs spinors in canonical layout (device), precision = 32 | 64 selects both the
 * arithmetic and the element type of in/out.  Asynchronous on `stream`.  in and out must not alias. */
int dslash_apply(clover_ctx *ctx, int op, int precision, const void *in_dev, void *out_dev, int n_rhs, void *stream);

/* Solve D psi_r = eta_r, r = 0..n_rhs-1, canonical fp64 in and out (device), by even-odd
 * preconditioned BiCGStab batched `batch` right-hand sides per Dslash launch (1, 2, 4 or 8, <= max_rhs):
 * mixed = 1: fp32 iteration with fp64 reliable updates (S 8(c) O6'); mixed = 0: everything fp64.
 * The iteration is the textbook recurrence with its dot products re-ordered (alpha from <Mhat^+ r0, p>, rho' from <r0,s> - omega <r0,t>;
 * DESIGN.md sec. 1) so that the BLAS-1 streams ride in the Dslash epilogues; results differ from the textbook ordering by rounding only.
 * Stops when the fp64 residual ||eta - D psi|| / ||eta|| <= tol (R10).  info_host: n_rhs entries, host.
 * Synchronises `stream`.  Returns the number of non-converged sources (0 = all good) or CLOVER_E*. */
int clover_solve(clover_ctx *ctx, const double *sources_dev, double *propagators_dev, int n_rhs, double tol,
                 int max_iter, int batch, int mixed, clover_rhs_info *info_host, void *stream);

/* Same, end to end from HOST buffers (pinned for full speed): batch i+1 is copied host -> device and the propagators of
 * batch i-1 device -> host on two internal copy streams while batch i is solved on `stream` (double-buffered device
 * staging owned by the context).  Work queued on `stream` before the call is waited for first; the call returns when
 * every propagator is in propagators_host.  At most 64 batches per call.  (Used for the e2e measurement.) */
int clover_solve_host(clover_ctx *ctx, const double *sources_host, double *propagators_host, int n_rhs, double tol,
                      int max_iter, int batch, int mixed, clover_rhs_info *info_host, void *stream);

/* Z4 noise sources (docs/NOISE.md): out_dev = n_rhs canonical spinors, precision 32 | 64,
 * source index r = rhs_offset + j; dilution: bit 0 keeps only timeslice t = r mod T, bit 1 keeps only the spin-colour
 * component (r / T, or r without the time bit) mod 12 ("time-spin-color dilution"); 0 = undiluted.
 * Needs no context.  Asynchronous on `stream`.  Bit-exact against the written spec. */
int noise_fill(void *out_dev, int precision, const int dims[4], uint64_t seed, int n_rhs, int rhs_offset,
               int dilution, double scale, void *stream);

/* ---- stochastic-operator contraction (S 8(f) rank 1; paper eqs. 7.5-7.7) ---- */
/* O_ij(t) = sum_y eta_i^*(t,y) gamma5 X_j(t,y)  (eq. 7.6: sum over the timeslice, spin and colour; gamma5 = diag(+,+,-,-) in the
 * basis R1).  eta_dev, x_dev: n_rhs canonical fp64 spinors each (device); o_dev: double [T][n_rhs][n_rhs][2] (device), index
 * [t][i][j].  fp64 arithmetic, deterministic summation order.  Needs no context; scratch is stream-ordered
 * (cudaMallocAsync).  Asynchronous on `stream`. */
int stochastic_operators(const double *eta_dev, const double *x_dev, const int dims[4], int n_rhs, double *o_dev, void *stream);
/* The same O_ij(t) (eq. 7.6) for callers that cannot allocate: code under CUDA graph capture, tight serving loops, harnesses
 * that forbid cudaMalloc.  This call allocates and frees NOTHING (no cudaMalloc / cudaMallocAsync / cudaFree): the per-chunk partial sums go to
 * a fixed 16 MiB device array inside the library (held by every GPU that loads it, until exit), so the size is limited:
 * T * n_rhs^2 <= CLOVER_NOALLOC_MAX_TNN, else CLOVER_EINVAL with a message (use stochastic_operators then).  Inputs and output as for
 * stochastic_operators, caller-owned.  All calls share the array and it keeps the last call's contents (nothing in it needs clearing: every
 * element read is written first by the same call); calls that OVERLAP on the GPU (two streams, two host threads) race on it -- serialise
 * them.  Results equal stochastic_operators up to the summation order over k-chunks (1e-13).  Asynchronous on `stream`. */
#define CLOVER_NOALLOC_MAX_TNN 1048576
int stochastic_operators_noalloc(const double *eta_dev, const double *x_dev, const int dims[4], int n_rhs, double *o_dev, void *stream);
/* C(t0, t) = (1 / (n_rhs^2 scale^4)) sum_ij O_ij(t) O_ji(t0)  (eq. 7.7 for every pair of timeslices; scale = the noise scale,
 * R7).  o_dev as above; c_dev: double [T][T][2] (device), index [t0][t].  Asynchronous on `stream`. */
int stochastic_correlator(const double *o_dev, int T, int n_rhs, double scale, double *c_dev, void *stream);

/* ---- outer-product fill (S 8(f) rank 2; paper eq. 7.3, Tables I-II "S_s fill", "S_s^dagger fill") ---- */
/* S(t,z,a; t0,x,b) = (1/(n_rhs scale^2)) sum_i X_i(t,z,a) conj(eta_i(t0,x,b)),  a, b = 3*spin + colour, z and x spatial sites in
 * canonical (z,y,x) order.  x_dev, eta_dev: n_rhs canonical fp64 spinors (device).  s_dev (device, caller-owned,
 * 12V x 12L^3 complex128 = 2304 T L^6 x 16 bytes): dagger = 0 -> double [T][L^3][12][L^3][12][2];
 * dagger = 1 -> the Hermitian conjugate, double [L^3][12][T][L^3][12][2].  All sources in one pass (the array is written once).
 * fp64.  Asynchronous on `stream`. */
int stochastic_fill(const double *x_dev, const double *eta_dev, const int dims[4], int n_rhs, int t0, double scale, int dagger,
                    double *s_dev, void *stream);

/* ---- trace operations of Table I (S 8(f) rank 3) ---- */
/* out[t] = sum_{o < n_outer} sum_{k < slice_len} |f[o][t][k]|^2 for a complex128 device field viewed as [n_outer][T][slice_len]:
 * with f = 12 point-source solutions (n_outer = 12, slice_len = 12 L^3) this is sum_y Tr[S_p(t,y;0,0) S_p^+(t,y;0,0)], the
 * zero-momentum pion correlator; with f = the array of stochastic_fill (n_outer = 1, slice_len = 144 L^6) it is
 * sum_x sum_z Tr[S_s(t,z;0,x) S_s^+(t,z;0,x)].  out_dev: double [T] (device).  fp64, deterministic.  Asynchronous on `stream`. */
int timeslice_norm2(const double *f_dev, long long n_outer, int T, long long slice_len, double *out_dev, void *stream);
/* out[t] = sum_{o, k} a[o][t][k] conj(b[o][t][k]) for two complex128 device fields of that shape: with a, b the arrays of two
 * stochastic_fill calls fed from INDEPENDENT source sets ("two sets of random sources, one for S and one for S^+", P:L303;
 * Figs. 2-3: no noise-squared bias, unlike the one-set trace) this is sum_x sum_z Tr[S_s^(1) S_s^(2)+](t).
 * out_dev: double [T][2] (device).  a_dev = b_dev gives (timeslice_norm2, 0).  fp64, deterministic.  Asynchronous on `stream`. */
int timeslice_inner(const double *a_dev, const double *b_dev, long long n_outer, int T, long long slice_len, double *out_dev, void *stream);

/* ---- measurement helpers (internal layout, no reorders; used by bench.py and the ncu runs) ---- */
enum {
    CLOVER_KERNEL_HOP = 0,        /* out_e = H_eo in_o                          (1320 flop/site)  */
    CLOVER_KERNEL_AINV_HOP = 1,   /* t_o = A_oo^-1 H_oe x_e                      (1824 flop/site) */
    CLOVER_KERNEL_A_MINUS_HOP = 2, /* y_e = A_ee x_e - kappa^2 H_eo t_o + <y,x>, <y,y>   (1872 flop/site) */
    /* the two variants the merged BiCGStab iteration launches (both also read a third field w at the own site): */
    CLOVER_KERNEL_A_MINUS_HOP_S = 3,  /* s_e = w_e - alpha (A_ee x_e - kappa^2 H_eo t_o), no reduction            */
    CLOVER_KERNEL_A_MINUS_HOP_XW = 4  /* y_e as in 2, + <w,y>, <w,x>                                                */
};
/* Launch one Dslash-type kernel `reps` times back to back on internal-layout scratch fields filled with
 * pseudo-random data and return the mean device time per launch in milliseconds (CUDA events on
 * `stream`).  precision 32 | 64; n_rhs in {1,2,4,8}.  flush_l2 != 0 writes a 256 MB buffer between
 * launches (outside the event pairs). */
int clover_bench_kernel(clover_ctx *ctx, int kernel, int precision, int n_rhs, int reps, int flush_l2, float *ms_per_launch,
                        void *stream);

/* Counters of the last clover_solve* call on this context: kernels launched, and device time (ms) spent
 * in the phases {reorder in/out, source prep, iteration, reliable updates, reconstruct+verify}, summed over batches. */
typedef struct {
    long long kernel_launches;
    double ms_total, ms_reorder, ms_prep, ms_iterate, ms_reliable, ms_finish;
    /* the two Dslash kernels of the sloppy (iteration-precision) Mhat, timed launch by launch with CUDA events on `stream`:
       ainv_hop = t_o = A_oo^-1 H_oe x_e ;  a_minus_hop = y_e = A_ee x_e - kappa^2 H_eo t_o with its dot-product epilogue */
    long long n_ainv_hop, n_a_minus_hop;
    double ms_ainv_hop, ms_a_minus_hop;
    /* merged iteration (default): the a_minus_hop launch of Mhat p that also writes s = r - alpha v is counted here, and
       n_a_minus_hop / ms_a_minus_hop count the one of Mhat s (with <t,s>, <t,t>, <r0,t>, <r0,s>) */
    long long n_a_minus_hop_s;
    double ms_a_minus_hop_s;
    /* merged iteration: the one BLAS-1 sweep of the iteration (x, r, p updates with <q0,p>, ||r||^2: 9 vector passes) */
    long long n_xrp_update;
    double ms_xrp_update;
} clover_solve_stats;
int clover_get_stats(const clover_ctx *ctx, clover_solve_stats *out);

/* Message for the last error on the calling thread (never NULL; ctx may be NULL). */
const char *clover_last_error(const clover_ctx *ctx);

#ifdef __cplusplus
}
#endif
#endif
