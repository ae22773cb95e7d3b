// blas.cuh -- host interface of the fused BLAS-1 / reduction / scalar kernels of the batched BiCGStab.
#pragma once
#include "context.h"

namespace clv {

// number of 16-byte vectors of a half-lattice field with B rhs
template <typename R> inline size_t field_vecs(const Geom &g, int B) { return (size_t)lb_blocks((unsigned)g.Vh * B) * 32u * Vec<R>::NV; }

struct BlasCtx {
    const Geom *g;
    int B;
    RhsScalars *sc;    // device, B entries
    double *partial;   // device, [blocks][B][4]
    double *partial2;  // device, same shape: second plane of the DOT_XW epilogue (merged iteration)
    int max_partial_blocks;
    double *stage;     // device, [8 rhs][32 slices][8]: second-level partials of the scalar kernels
    unsigned *ticket;  // device, [8]: arrival counters of the scalar kernels (zero between launches)
    cudaStream_t st;
    long long *launches;
    double brk2;       // square of the relative breakdown threshold of the iteration precision (scalar kernel, R11)
};

// s = r - alpha v
template <typename R> int blas_s_update(const BlasCtx &c, const typename Vec<R>::T *r, const typename Vec<R>::T *v, typename Vec<R>::T *s);
// x += alpha p + omega s ; r = s - omega t ; partial <r0,r>, ||r||^2 ; returns number of partial blocks
template <typename R>
int blas_xr_update(const BlasCtx &c, typename Vec<R>::T *x, typename Vec<R>::T *r, const typename Vec<R>::T *p, const typename Vec<R>::T *s,
                   const typename Vec<R>::T *t, const typename Vec<R>::T *r0, int *nblocks);
// p = r + beta (p - omega v)
template <typename R> int blas_p_update(const BlasCtx &c, typename Vec<R>::T *p, const typename Vec<R>::T *r, const typename Vec<R>::T *v);
// y += x (fp64 accumulate), x = 0
template <typename R> int blas_accumulate_y(const BlasCtx &c, double2 *y, typename Vec<R>::T *x);
// r64 = b - w (w may be null: r64 = b; r64 itself may be null: not stored) ; rs = (R) r64 ; partial ||r64||^2
template <typename R> int blas_residual(const BlasCtx &c, const double2 *b, const double2 *w, double2 *r64, typename Vec<R>::T *rs, int *nblocks);
// partial d0 = ||a1 - b1||^2, d1 = ||a2 - b2||^2 (b1, b2 may be null)
int blas_norm2_pair(const BlasCtx &c, const double2 *a1, const double2 *b1, const double2 *a2, const double2 *b2, int *nblocks);

// scalar steps (one block per rhs): reduce the partials of `nblocks` blocks and update RhsScalars
enum { SC_ETA2 = 0, SC_INIT = 1, SC_ALPHA = 2, SC_OMEGA = 3, SC_RHO = 4, SC_TRUE = 5, SC_FINAL = 6, SC_RESTART = 7,
       SC_INIT_MERGED = 8, SC_OMEGA2 = 9, SC_RHO2 = 10, SC_RESTART2 = 11,  // merged iteration (solver.cu)
       SC_CONFIRM = 12 };  // full-lattice verification that also decides convergence
// r0 = r for the rhs whose `restart` flag is set (breakdown recovery)
template <typename R> int blas_restart(const BlasCtx &c, const typename Vec<R>::T *r, typename Vec<R>::T *r0, typename Vec<R>::T *p = nullptr);
// merged iteration: x += alpha p + omega s ; r' = s - omega t ; p = r' + beta p - gam (r - s) ; partial <q0,p>, ||r'||^2
template <typename R>
int blas_xrp_update(const BlasCtx &c, typename Vec<R>::T *x, typename Vec<R>::T *r, typename Vec<R>::T *p, const typename Vec<R>::T *s,
                    const typename Vec<R>::T *t, const typename Vec<R>::T *q0, int *nblocks);
// out = gamma5 in (masked: only the rhs flagged restart == 1 are written)
template <typename R> int blas_gamma5(const BlasCtx &c, const typename Vec<R>::T *in, typename Vec<R>::T *out, int masked);
// partial <a, b>
template <typename R> int blas_cdot(const BlasCtx &c, const typename Vec<R>::T *a, const typename Vec<R>::T *b, int *nblocks);
// `publish` (device address of mapped pinned host memory, B entries) != nullptr: each rhs' scalars are also stored there
int blas_scalar_step(const BlasCtx &c, int step, int nblocks, double tol2, double delta2, RhsScalars *publish = nullptr);

}  // namespace clv
