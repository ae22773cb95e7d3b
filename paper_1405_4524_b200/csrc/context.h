// context.h -- the opaque clover_ctx and the internal (host-side) interfaces between translation units.
#pragma once
#include "../../include/clover.h"
#include "common.cuh"
#include <vector>

namespace clv {

// Per-precision operator data in the internal layout (device pointers owned by the context).
template <typename R> struct OpData {
    typedef typename Vec<R>::C C;
    C *gauge[2][4];   // [parity of the site the link lives at][mu], lane-blocked over cb, NK = recon/2
    C *clov[2];       // A   : [parity], 36 complex per site (2 blocks x (3 packed diag pairs + 15 lower off-diag))
    C *clov_inv[2];   // A^-1, same packing
    int recon;        // 18 | 12
    // Site-major ("packed") copies for the B = 8 kernels, fetched per CTA tile with one bulk async copy each (dslash3_kernel.cuh):
    // Records are padded (pk_link_stride / PK_CLOV_STRIDE reals per site) so that in shared memory the 8 sites of a warp tile fall into
    // disjoint 4-bank groups: a warp-wide 16-byte load of "the same element of 8 sites" is then one conflict-free wavefront.
    R *pk_link[2];     // [parity p of the OUTPUT site][cb][d = 2 mu + (fwd ? 0 : 1)][recon reals]: fwd = U_mu(x), bwd = U_mu(x - mu) as stored
    R *pk_clov[2];     // [parity][cb][72 reals]: the 18 16-byte rows (fp32) of the packed blocks of A
    R *pk_clov_inv[2]; // A^-1
};
// reals per site record: 8 links of `recon` reals + 4 of padding (592 or 400 bytes in fp32: 20 s or 4 s words mod 32 for site s), 72 + 4 for the clover blocks
#ifndef CLV_PK_PAD
#define CLV_PK_PAD 4
#endif
__host__ __device__ constexpr int pk_link_stride(int recon) { return 8 * recon + CLV_PK_PAD; }
constexpr int PK_CLOV_STRIDE = 72 + CLV_PK_PAD;

// Per-rhs solver scalars, device resident (one entry per rhs of the batch).
struct RhsScalars {
    double2 rho, alpha, omega, beta;  // BiCGStab recurrences (complex)
    double2 gam;      // merged iteration: rho'/rho = beta omega / alpha, the coefficient of (r - s) = alpha v in the p update
    double r2;        // ||r||^2 of the iterated (sloppy) residual
    double maxr2;     // max ||r||^2 since the last reliable update
    double eta2;      // ||eta||^2 on the full lattice (stopping scale, R10)
    double true_r2;   // ||r||^2 at the last fp64 recomputation
    int done;         // 1 once the fp64 residual met the tolerance (rhs frozen)
    int want_update;  // 1 if this rhs asks for a reliable update (||r|| < delta max||r||, or stagnation)
    int status;       // clover_rhs_info.status
    int claim;        // 1 if the iterated residual of this rhs meets the tolerance (to be confirmed in fp64)
    int restart;      // 1 if <r0, v> vanished this iteration: r0 := r, rho := ||r||^2 before the next one (R11)
    int nrestart;     // restarts so far (a rhs that keeps breaking down ends with status 2)
    // reliable-update control of this rhs (R11): a leg of sloppy iterations ends when ||r||^2 < delta2 * max||r||^2, or after LEG_MAX
    // iterations.  delta2 starts at the solver's delta^2 and is RAISED when a reliable update finds the true residual well above the
    // iterated one (the leg asked the sloppy precision for more than it can deliver: ill-conditioned systems), so that the next legs
    // stop where the sloppy residual is still true.
    double delta2;
    double r0n2;      // ||r0||^2 at the last (re)start: scale of the relative breakdown test |<r0, r>| <= brk ||r0|| ||r|| (R11)
    int since;        // sloppy iterations since the last reliable update
    int pad_;
};

struct SolveWork;  // solver.cu

}  // namespace clv

struct clover_ctx {
    clv::Geom geom;
    double kappa, csw;
    int max_rhs;
    clv::OpData<double> op64;
    clv::OpData<float> op32;
    // scratch fields (internal layout) sized for max_rhs, allocated lazily by the solver / bench / dslash_apply
    clv::SolveWork *work;
    clover_solve_stats stats;
    unsigned *sched;             // two device counters (zeroed) of the persistent Dslash kernels' tile scheduler; they leave them zeroed
    std::vector<void *> allocs;  // every device allocation of the operator data (freed by clover_destroy)
};

namespace clv {

// ---- setup.cu ----
int setup_operator(clover_ctx *ctx, const double *gauge_dev, cudaStream_t st);
// canonical <-> internal reorders; CT = element type of the canonical array, R = internal real type.
// canon: [n_rhs][V][12] complex of CT; even/odd: internal fields with B = n_rhs.
template <typename CT, typename R>
int reorder_in(const Geom &g, const CT *canon, typename Vec<R>::T *even, typename Vec<R>::T *odd, int B, cudaStream_t st);
template <typename CT, typename R>
int reorder_out(const Geom &g, CT *canon, const typename Vec<R>::T *even, const typename Vec<R>::T *odd, int B, cudaStream_t st);

// ---- dslash.cu ----
// out = P ( X + coef * H_{p,1-p} in ),  P = 1 | A_pp^-1,  X = 0 | xin | A_pp xin   (p = parity of out)
enum { XM_NONE = 0, XM_PLAIN = 1, XM_CLOVER = 2 };
// DOT_S / DOT_XW are the epilogues of the merged BiCGStab iteration (solver.cu): DOT_S computes v = (...) but stores only s = w - alpha v
// (to `out2`; `out` is not written) (alpha = sc[rhs].alpha, already known when the kernel starts; no reduction); DOT_XW is DOT_X plus <w, out> and <w, xin>.
enum { DOT_NONE = 0, DOT_W = 1, DOT_X = 2, DOT_RES = 3, DOT_S = 4, DOT_XW = 5 };
template <typename R> struct DslashArgs {
    typedef typename Vec<R>::T V;
    const V *in;      // parity 1-p field
    const V *xin;     // parity p field (XM_PLAIN / XM_CLOVER)
    V *out;           // parity p field
    const V *w;       // DOT_W: partial <w, out> per rhs.  DOT_RES: the result is w - (...), partial ||result||^2
    float4 *out32;    // DOT_RES only: if non-null the result is stored here in fp32 instead of `out` (reliable update: r = b - Mhat y)
    double *partial;  // [gridDim.x][B][4] : DOT_W -> (re,im of <w,out>, 0, 0); DOT_X -> (re,im of <out,xin>, <out,out>, 0)
    double *partial2; // DOT_XW: second plane, same shape: (re,im of <w,out>, re,im of <w,xin>)
    V *out2;          // DOT_S: s = w - alpha * result (the only store of that variant)
    const RhsScalars *sc;  // DOT_S: per-rhs scalars (alpha)
    R coef;
    int parity;       // p
    int xmode, pinv, dot;
};
template <typename R> int launch_dslash(const clover_ctx *ctx, const DslashArgs<R> &a, int B, cudaStream_t st, int *grid_out);
// out = A in or A^-1 in on one parity
template <typename R>
int launch_clover(const clover_ctx *ctx, const typename Vec<R>::T *in, typename Vec<R>::T *out, int parity, int inverse, int B,
                  cudaStream_t st);
int dslash_block_size();

// ---- noise.cu ----
int launch_noise(void *out, int precision, const int dims[4], uint64_t seed, int n_rhs, int rhs_offset, int dilution, double scale,
                 cudaStream_t st);

// ---- contract.cu ----
int launch_contract(const double *eta, const double *xs, const int dims[4], int n, double *o, cudaStream_t st);
int launch_contract_noalloc(const double *eta, const double *xs, const int dims[4], int n, double *o, cudaStream_t st);
int launch_correlator(const double *o, int T, int n, double scale, double *c, cudaStream_t st);

// ---- fill.cu ----
int launch_fill(const double *x, const double *eta, const int dims[4], int n, int t0, double scale, int dagger, double *s, cudaStream_t st);

// ---- traces.cu ----
int launch_timeslice_norm2(const double *f, long n_outer, int T, long slice_len, double *out, cudaStream_t st);
int launch_timeslice_inner(const double *a, const double *b, long n_outer, int T, long slice_len, double *out, cudaStream_t st);

// ---- solver.cu ----
int solve_batches(clover_ctx *ctx, const double *src, double *dst, int n_rhs, double tol, int max_iter, int batch, int mixed,
                  clover_rhs_info *info, cudaStream_t st, int host_buffers);
void free_work(clover_ctx *ctx);
int bench_kernel(clover_ctx *ctx, int kernel, int precision, int n_rhs, int reps, int flush_l2, float *ms, cudaStream_t st);
int apply_op(clover_ctx *ctx, int op, int precision, const void *in, void *out, int n_rhs, cudaStream_t st);

}  // namespace clv
