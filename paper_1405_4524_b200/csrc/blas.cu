// blas.cu -- fused BLAS-1 updates, deterministic two-stage reductions and the per-rhs scalar recurrences of the
// batched BiCGStab (SURVEY 8(a) H5, 8(c) O6').  Fields are lane-blocked (common.cuh): vector i of a field belongs
// to rhs = i & (B-1), so every kernel is a flat, fully coalesced sweep over 16-byte vectors.
// Reductions: products in the storage precision, accumulation in fp64, warp shuffle -> shared memory ->
// per-block partials [block][rhs][4]; the scalar kernels sum the partials in a fixed order (deterministic).
#include "blas.cuh"
#include <cstdlib>
#include <algorithm>

namespace clv {

constexpr int BLAS_BLOCK = 256;
constexpr int BLAS_MAX_GRID = 148 * 8;

// ---- complex helpers on 16-byte vectors -----------------------------------------------------------
struct zs {
    double re, im;
};  // a complex scalar
__device__ __forceinline__ zs ld_z(const double2 &v) { return zs{v.x, v.y}; }

// a + z*b  (per complex component of the vector)
__device__ __forceinline__ float4 caxpy(zs z, float4 b, float4 a)
{
    const float zr = (float)z.re, zi = (float)z.im;
    a.x += zr * b.x - zi * b.y;
    a.y += zr * b.y + zi * b.x;
    a.z += zr * b.z - zi * b.w;
    a.w += zr * b.w + zi * b.z;
    return a;
}
__device__ __forceinline__ double2 caxpy(zs z, double2 b, double2 a)
{
    a.x += z.re * b.x - z.im * b.y;
    a.y += z.re * b.y + z.im * b.x;
    return a;
}
__device__ __forceinline__ zs neg(zs z) { return zs{-z.re, -z.im}; }
// conj(a) . b accumulated in fp64, |a|^2
__device__ __forceinline__ void cdot_acc(float4 a, float4 b, double &re, double &im)
{
    re += (double)(a.x * b.x + a.y * b.y + a.z * b.z + a.w * b.w);
    im += (double)(a.x * b.y - a.y * b.x + a.z * b.w - a.w * b.z);
}
__device__ __forceinline__ void cdot_acc(double2 a, double2 b, double &re, double &im)
{
    re += a.x * b.x + a.y * b.y;
    im += a.x * b.y - a.y * b.x;
}
__device__ __forceinline__ double norm2(float4 a) { return (double)(a.x * a.x + a.y * a.y + a.z * a.z + a.w * a.w); }
__device__ __forceinline__ double norm2(double2 a) { return a.x * a.x + a.y * a.y; }

// block reduction with runtime B (B | 32); partial[(block*B + rhs)*4 + c]
__device__ __forceinline__ void block_reduce(int B, double v0, double v1, double v2, double *__restrict__ partial)
{
    __shared__ double sm[BLAS_BLOCK / 32][8][3];
    for (int off = 16; off >= B; off >>= 1) {
        v0 += __shfl_xor_sync(0xffffffffu, v0, off);
        v1 += __shfl_xor_sync(0xffffffffu, v1, off);
        v2 += __shfl_xor_sync(0xffffffffu, v2, off);
    }
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (lane < B) {
        sm[warp][lane][0] = v0;
        sm[warp][lane][1] = v1;
        sm[warp][lane][2] = v2;
    }
    __syncthreads();
    if ((int)threadIdx.x < B * 3) {
        const int r = threadIdx.x / 3, c = threadIdx.x % 3;
        double s = 0;
        for (int w = 0; w < BLAS_BLOCK / 32; w++) s += sm[w][r][c];
        partial[((size_t)blockIdx.x * B + r) * 4 + c] = s;
    }
}

static inline int blas_grid(size_t nvec) { return (int)std::min<size_t>((nvec + BLAS_BLOCK - 1) / BLAS_BLOCK, BLAS_MAX_GRID); }

// ---- s = r - alpha v --------------------------------------------------------------------------------
template <typename V> __global__ void __launch_bounds__(BLAS_BLOCK) s_update_kernel(size_t n, int B, const RhsScalars *__restrict__ sc,
                                                                                     const V *__restrict__ r, const V *__restrict__ v, V *__restrict__ s)
{
    const zs ma = neg(ld_z(sc[threadIdx.x & (B - 1)].alpha));
    for (size_t i = (size_t)blockIdx.x * BLAS_BLOCK + threadIdx.x; i < n; i += (size_t)gridDim.x * BLAS_BLOCK) s[i] = caxpy(ma, v[i], r[i]);
}

// ---- x += alpha p + omega s ; r = s - omega t ; <r0,r>, ||r||^2 ----------------------------------------
template <typename V>
__global__ void __launch_bounds__(BLAS_BLOCK) xr_update_kernel(size_t n, int B, const RhsScalars *__restrict__ sc, V *__restrict__ x, V *__restrict__ r,
                                                               const V *__restrict__ p, const V *__restrict__ s, const V *__restrict__ t,
                                                               const V *__restrict__ r0, double *__restrict__ partial)
{
    const RhsScalars &q = sc[threadIdx.x & (B - 1)];
    const zs al = ld_z(q.alpha), om = ld_z(q.omega), mom = neg(om);
    double d0 = 0, d1 = 0, d2 = 0;
    for (size_t i = (size_t)blockIdx.x * BLAS_BLOCK + threadIdx.x; i < n; i += (size_t)gridDim.x * BLAS_BLOCK) {
        const V sv = s[i];
        x[i] = caxpy(om, sv, caxpy(al, p[i], x[i]));
        const V rn = caxpy(mom, t[i], sv);
        r[i] = rn;
        cdot_acc(r0[i], rn, d0, d1);
        d2 += norm2(rn);
    }
    block_reduce(B, d0, d1, d2, partial);
}

// ---- r0 = r for the rhs flagged `restart` ------------------------------------------------------------
template <typename V> __global__ void __launch_bounds__(BLAS_BLOCK) restart_kernel(size_t n, int B, const RhsScalars *__restrict__ sc, const V *__restrict__ r,
                                                                                    V *__restrict__ r0, V *__restrict__ p)
{
    if (sc[threadIdx.x & (B - 1)].restart != 1) return;
    for (size_t i = (size_t)blockIdx.x * BLAS_BLOCK + threadIdx.x; i < n; i += (size_t)gridDim.x * BLAS_BLOCK) {
        const V a = r[i];
        r0[i] = a;
        if (p) p[i] = a;   // merged iteration: the search direction restarts with the shadow residual
    }
}

// ---- p = r + beta (p - omega v) ---------------------------------------------------------------------
template <typename V> __global__ void __launch_bounds__(BLAS_BLOCK) p_update_kernel(size_t n, int B, const RhsScalars *__restrict__ sc, V *__restrict__ p,
                                                                                     const V *__restrict__ r, const V *__restrict__ v)
{
    const RhsScalars &q = sc[threadIdx.x & (B - 1)];
    const zs be = ld_z(q.beta), mom = neg(ld_z(q.omega));
    for (size_t i = (size_t)blockIdx.x * BLAS_BLOCK + threadIdx.x; i < n; i += (size_t)gridDim.x * BLAS_BLOCK) p[i] = caxpy(be, caxpy(mom, v[i], p[i]), r[i]);
}

// ---- merged iteration (solver.cu): x += alpha p + omega s ; r' = s - omega t ; p = r' + beta p - gam (r - s) ; <q0,p>, ||r'||^2.
//      (r - s = alpha v and gam = beta omega / alpha, so this is p = r' + beta (p - omega v) without v ever being stored.) ----
__device__ __forceinline__ float4 vsub(float4 a, float4 b) { return make_float4(a.x - b.x, a.y - b.y, a.z - b.z, a.w - b.w); }
__device__ __forceinline__ double2 vsub(double2 a, double2 b) { return make_double2(a.x - b.x, a.y - b.y); }
template <typename V>
__global__ void __launch_bounds__(BLAS_BLOCK) xrp_update_kernel(size_t n, int B, const RhsScalars *__restrict__ sc, V *__restrict__ x, V *__restrict__ r,
                                                                V *__restrict__ p, const V *__restrict__ s, const V *__restrict__ t,
                                                                const V *__restrict__ q0, double *__restrict__ partial)
{
    const RhsScalars &q = sc[threadIdx.x & (B - 1)];
    const zs al = ld_z(q.alpha), om = ld_z(q.omega), mom = neg(om), be = ld_z(q.beta), mga = neg(ld_z(q.gam));
    double d0 = 0, d1 = 0, d2 = 0;
    for (size_t i = (size_t)blockIdx.x * BLAS_BLOCK + threadIdx.x; i < n; i += (size_t)gridDim.x * BLAS_BLOCK) {
        const V sv = s[i], pv = p[i], ro = r[i];
        x[i] = caxpy(om, sv, caxpy(al, pv, x[i]));
        const V rn = caxpy(mom, t[i], sv);
        r[i] = rn;
        const V pn = caxpy(mga, vsub(ro, sv), caxpy(be, pv, rn));
        p[i] = pn;
        cdot_acc(q0[i], pn, d0, d1);
        d2 += norm2(rn);
    }
    block_reduce(B, d0, d1, d2, partial);
}

// ---- out = gamma5 in (chiral basis: spins 2, 3 change sign = the upper half of the NV vectors of an entry);
//      `masked`: only the rhs flagged `restart == 1` are written ------------------------------------------------
__device__ __forceinline__ float4 vneg(float4 a) { return make_float4(-a.x, -a.y, -a.z, -a.w); }
__device__ __forceinline__ double2 vneg(double2 a) { return make_double2(-a.x, -a.y); }
template <typename V, int NV>
__global__ void __launch_bounds__(BLAS_BLOCK) gamma5_kernel(size_t n, int B, const RhsScalars *__restrict__ sc, int masked, const V *__restrict__ in,
                                                            V *__restrict__ out)
{
    if (masked && sc[threadIdx.x & (B - 1)].restart != 1) return;
    for (size_t i = (size_t)blockIdx.x * BLAS_BLOCK + threadIdx.x; i < n; i += (size_t)gridDim.x * BLAS_BLOCK) {
        const V a = in[i];
        out[i] = ((i >> 5) % NV >= NV / 2) ? vneg(a) : a;
    }
}

// ---- partial <a, b> -----------------------------------------------------------------------------------
template <typename V>
__global__ void __launch_bounds__(BLAS_BLOCK) cdot_kernel(size_t n, int B, const V *__restrict__ a, const V *__restrict__ b, double *__restrict__ partial)
{
    double d0 = 0, d1 = 0;
    for (size_t i = (size_t)blockIdx.x * BLAS_BLOCK + threadIdx.x; i < n; i += (size_t)gridDim.x * BLAS_BLOCK) cdot_acc(a[i], b[i], d0, d1);
    block_reduce(B, d0, d1, 0., partial);
}

// ---- y += x ; x = 0.  fp32 x: vector (jb, k, lane) holds the complex numbers 2k, 2k+1 = fp64 vectors (jb, 2k), (jb, 2k+1) ----
__global__ void __launch_bounds__(BLAS_BLOCK) accumulate_y_kernel(size_t n32, double2 *__restrict__ y, float4 *__restrict__ x)
{
    for (size_t i = (size_t)blockIdx.x * BLAS_BLOCK + threadIdx.x; i < n32; i += (size_t)gridDim.x * BLAS_BLOCK) {
        const size_t lane = i & 31, row = i >> 5;  // row = jb*6 + k
        const size_t jb = row / 6, k = row % 6;
        const size_t o = ((jb * 12 + 2 * k) << 5) + lane;
        const float4 v = x[i];
        double2 a = y[o], b = y[o + 32];
        a.x += (double)v.x; a.y += (double)v.y;
        b.x += (double)v.z; b.y += (double)v.w;
        y[o] = a;
        y[o + 32] = b;
        x[i] = make_float4(0.f, 0.f, 0.f, 0.f);
    }
}
__global__ void __launch_bounds__(BLAS_BLOCK) accumulate_y_kernel(size_t n64, double2 *__restrict__ y, double2 *__restrict__ x)
{
    for (size_t i = (size_t)blockIdx.x * BLAS_BLOCK + threadIdx.x; i < n64; i += (size_t)gridDim.x * BLAS_BLOCK) {
        double2 a = y[i];
        const double2 v = x[i];
        a.x += v.x; a.y += v.y;
        y[i] = a;
        x[i] = make_double2(0., 0.);
    }
}

// ---- r64 = b - w ; rs = (R) r64 ; ||r64||^2.  Indexed by the fp64 vector index. -------------------------
__device__ __forceinline__ void store_sloppy(float4 *rs, size_t i, double2 v)
{
    // fp64 vector (jb, kk, lane) -> half of fp32 vector (jb, kk/2, lane)
    const size_t lane = i & 31, row = i >> 5, jb = row / 12, kk = row % 12;
    float2 *dst = reinterpret_cast<float2 *>(rs + (((jb * 6 + (kk >> 1)) << 5) + lane)) + (kk & 1);
    *dst = make_float2((float)v.x, (float)v.y);
}
__device__ __forceinline__ void store_sloppy(double2 *rs, size_t i, double2 v) { rs[i] = v; }

template <typename V>
__global__ void __launch_bounds__(BLAS_BLOCK) residual_kernel(size_t n64, int B, const double2 *__restrict__ b, const double2 *__restrict__ w,
                                                              double2 *__restrict__ r64, V *__restrict__ rs, double *__restrict__ partial)
{
    double d0 = 0;
    for (size_t i = (size_t)blockIdx.x * BLAS_BLOCK + threadIdx.x; i < n64; i += (size_t)gridDim.x * BLAS_BLOCK) {
        double2 v = b[i];
        if (w) {
            const double2 ww = w[i];
            v.x -= ww.x;
            v.y -= ww.y;
        }
        if (r64) r64[i] = v;
        store_sloppy(rs, i, v);
        d0 += norm2(v);
    }
    block_reduce(B, d0, 0., 0., partial);
}

// ---- d0 = ||a1 - b1||^2, d1 = ||a2 - b2||^2 (b1, b2 may be null) --------------------------------------------
__device__ __forceinline__ double diff2(const double2 *__restrict__ a, const double2 *__restrict__ b, size_t i)
{
    double2 v = a[i];
    if (b) {
        const double2 bb = b[i];
        v.x -= bb.x;
        v.y -= bb.y;
    }
    return norm2(v);
}
__global__ void __launch_bounds__(BLAS_BLOCK) norm2_pair_kernel(size_t n64, int B, const double2 *__restrict__ a1, const double2 *__restrict__ b1,
                                                                const double2 *__restrict__ a2, const double2 *__restrict__ b2,
                                                                double *__restrict__ partial)
{
    double d0 = 0, d1 = 0;
    for (size_t i = (size_t)blockIdx.x * BLAS_BLOCK + threadIdx.x; i < n64; i += (size_t)gridDim.x * BLAS_BLOCK) {
        d0 += diff2(a1, b1, i);
        d1 += diff2(a2, b2, i);
    }
    block_reduce(B, d0, d1, 0., partial);
}

// ---- scalar steps -----------------------------------------------------------------------------------------
__device__ __forceinline__ zs zdiv(zs a, zs b)
{
    const double d = b.re * b.re + b.im * b.im;
    return zs{(a.re * b.re + a.im * b.im) / d, (a.im * b.re - a.re * b.im) / d};
}
__device__ __forceinline__ zs zmul(zs a, zs b) { return zs{a.re * b.re - a.im * b.im, a.re * b.im + a.im * b.re}; }
__device__ __forceinline__ double2 st_z(zs z) { return make_double2(z.re, z.im); }
__device__ __forceinline__ bool finite_z(zs z) { return isfinite(z.re) && isfinite(z.im); }

// one block per rhs: sum partial[(b*B + rhs)*4 + c] over b < nblocks in a fixed order, then thread 0 updates the scalars.
constexpr int SC_SLICES = 32;
constexpr int MAX_RESTARTS = 100;   // breakdown restarts of one rhs before it is given up (status 2)
constexpr int LEG_MAX = 48;   // sloppy iterations between two reliable updates at most (the benchmarked systems need 12-14 per leg)
__global__ void __launch_bounds__(256) scalar_kernel(int step, int B, int nblocks, const double *__restrict__ partial, const double *__restrict__ partial2,
                                                     RhsScalars *sc, double tol2, double delta2, double *stage, unsigned *ticket, RhsScalars *publish, int leg_max, double brk2)
{
    __shared__ double sm[256][7];
    __shared__ bool last;
    const int rhs = blockIdx.x, slice = blockIdx.y;
    // stage 1: this block sums its contiguous slice of the per-block partials (fixed order); plane 2 only where the step has one
    const int per = (nblocks + SC_SLICES - 1) / SC_SLICES, lo = slice * per, hi = min(nblocks, lo + per);
    double a[7] = {0, 0, 0, 0, 0, 0, 0};
    // (16-byte loads, four lines in flight per thread: the persistent B = 8 kernels leave one line per tile, 41472 at 24^3x48)
#pragma unroll 4
    for (int b = lo + threadIdx.x; b < hi; b += 256) {
        const double2 *q = reinterpret_cast<const double2 *>(partial + ((size_t)b * B + rhs) * 4);
        const double2 q01 = __ldcg(q), q23 = __ldcg(q + 1);
        a[0] += q01.x;
        a[1] += q01.y;
        a[2] += q23.x;
        if (partial2) {
            const double2 *q2 = reinterpret_cast<const double2 *>(partial2 + ((size_t)b * B + rhs) * 4);
            const double2 p01 = __ldcg(q2), p23 = __ldcg(q2 + 1);
            a[3] += p01.x;
            a[4] += p01.y;
            a[5] += p23.x;
            a[6] += p23.y;
        }
    }
#pragma unroll
    for (int c = 0; c < 7; c++) sm[threadIdx.x][c] = a[c];
    __syncthreads();
    for (int s = 128; s > 0; s >>= 1) {
        if ((int)threadIdx.x < s) {
#pragma unroll
            for (int c = 0; c < 7; c++) sm[threadIdx.x][c] += sm[threadIdx.x + s][c];
        }
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        double *o = stage + ((size_t)rhs * SC_SLICES + slice) * 8;
#pragma unroll
        for (int c = 0; c < 7; c++) o[c] = sm[0][c];
        __threadfence();
        last = (atomicAdd(ticket + rhs, 1u) == SC_SLICES - 1);
    }
    __syncthreads();
    if (!last || threadIdx.x >= 32) return;
    // stage 2 (last block of this rhs to arrive): lane k fetches slice k (one L2 round trip for all 32 slices instead of 32
    // dependent ones), a butterfly sums them in a fixed order, then lane 0 runs the scalar recurrences
    __threadfence();
    static_assert(SC_SLICES == 32, "one slice per lane");
    double e[7];
    {
        const volatile double *o = stage + ((size_t)rhs * SC_SLICES + threadIdx.x) * 8;
#pragma unroll
        for (int c = 0; c < 7; c++) e[c] = o[c];
    }
#pragma unroll
    for (int off = 16; off >= 1; off >>= 1) {
#pragma unroll
        for (int c = 0; c < 7; c++) e[c] += __shfl_xor_sync(0xffffffffu, e[c], off);
    }
    if (threadIdx.x != 0) return;
    ticket[rhs] = 0;
    const double d0 = e[0], d1 = e[1], d2 = e[2], e0 = e[3], e1 = e[4], e2 = e[5], e3 = e[6];
    RhsScalars &q = sc[rhs];
    const zs zero{0., 0.};
    switch (step) {
    case SC_ETA2:  // d0 = ||eta_e||^2, d1 = ||eta_o||^2
        q.eta2 = d0 + d1;
        q.done = 0;
        q.status = 0;
        q.want_update = 0;
        break;
    case SC_INIT:  // d0 = ||r||^2 with r = b_e (y = 0)
    case SC_INIT_MERGED:
        q.rho = make_double2(d0, 0.);
        q.r2 = q.maxr2 = q.true_r2 = d0;
        q.alpha = q.omega = q.beta = q.gam = make_double2(0., 0.);
        q.want_update = 0;
        q.claim = 0;
        q.restart = 0;
        q.nrestart = 0;
        q.delta2 = delta2;
        q.r0n2 = d0;   // r0 = r = b
        q.since = 0;
        if (!(q.eta2 > 0.) || d0 <= tol2 * q.eta2) q.done = 1;  // zero source or already converged
        if (!isfinite(d0)) { q.done = 1; q.status = 3; }
        if (step == SC_INIT_MERGED && !q.done) q.restart = 1;  // merged iteration: the start is a restart of every active rhs (SC_RESTART2)
        break;
    case SC_ALPHA: {  // (d0,d1) = <r0, v>
        zs al = zero;
        if (!q.done) {
            const zs r0v{d0, d1};
            if (!finite_z(r0v)) { q.done = 1; q.status = 3; }
            else if (!(d0 * d0 + d1 * d1 > 0.)) {
                // breakdown (e.g. a point source on unit links): this iteration becomes a pure minimal-residual step (alpha = 0),
                // then the recurrence restarts from the current residual, r0 := r (same remedy as the oracle, R11)
                if (q.nrestart < MAX_RESTARTS) { q.restart = 1; q.nrestart++; }
                else { q.done = 1; q.status = 2; }
            } else {
                al = zdiv(ld_z(q.rho), r0v);
                if (!finite_z(al)) { al = zero; if (q.nrestart < MAX_RESTARTS) { q.restart = 1; q.nrestart++; } else { q.done = 1; q.status = 2; } }
            }
        }
        q.alpha = st_z(al);
        break;
    }
    case SC_OMEGA: {  // (d0,d1) = <t, s>, d2 = <t, t>
        zs om = zero;
        if (!q.done) {
            if (!isfinite(d2) || !isfinite(d0) || !isfinite(d1)) { q.done = 1; q.status = 3; q.alpha = st_z(zero); }
            else if (d2 > 0.) om = zs{d0 / d2, d1 / d2};
        }
        q.omega = st_z(om);
        break;
    }
    case SC_RHO: {  // (d0,d1) = <r0, r>, d2 = ||r||^2
        zs be = zero;
        q.want_update = 0;
        q.claim = 0;
        if (!q.done) {
            const zs rho1{d0, d1}, om = ld_z(q.omega), rho = ld_z(q.rho);
            q.r2 = d2;
            if (d2 > q.maxr2) q.maxr2 = d2;
            if (!isfinite(d2) || !finite_z(rho1)) { q.done = 1; q.status = 3; }
            else {
                if (d2 < q.delta2 * q.maxr2 || ++q.since >= leg_max) q.want_update = 1;
                q.claim = (d2 <= tol2 * q.eta2) ? 1 : 0;
                const double om2 = om.re * om.re + om.im * om.im, rh2 = rho.re * rho.re + rho.im * rho.im;
                if (!(om2 > 0.) || !(rh2 > 0.)) q.want_update = 1;  // stagnation: let the fp64 residual decide, beta = 0 restarts p = r
                else be = zmul(zdiv(rho1, rho), zdiv(ld_z(q.alpha), om));
                if (!finite_z(be)) be = zero;
                // relative breakdown (as in the oracle): r0 has become orthogonal to r within the precision of the dot product -- restart the
                // recurrence from the current residual (r0 := r, p := r: beta = 0) rather than divide by a rho that is noise
                if (d2 > 0. && !q.restart && d0 * d0 + d1 * d1 <= brk2 * q.r0n2 * d2 && q.nrestart < MAX_RESTARTS) { q.restart = 1; q.nrestart++; be = zero; }
                q.rho = st_z(rho1);
            }
        }
        q.beta = st_z(be);
        break;
    }
    case SC_TRUE:  // d0 = ||b - Mhat y||^2 in fp64
        q.true_r2 = d0;
        q.claim = 0;
        if (!q.done) {
            // The leg that just ended started at max||r||^2 = maxr2 and claims the iterated q.r2.  If the true residual is more than twice the
            // claim, the sloppy precision gave out before the leg's target: ask the next legs for no more than four times (in ||r||) what
            // this one really achieved, never for less than a factor 10, never for more than the solver's delta.
            if (isfinite(d0) && d0 > 4. * q.r2 && q.maxr2 > 0.) q.delta2 = fmin(1e-2, fmax(q.delta2, 16. * d0 / q.maxr2));
            q.since = 0;
            q.r2 = q.maxr2 = d0;
            q.want_update = 0;
            if (!isfinite(d0)) { q.done = 1; q.status = 3; }
            // freeze on a bound 1 % inside the tolerance: the status is decided later on the full-lattice residual (SC_FINAL), which
            // equals this even-odd one only up to rounding, and a frozen rhs gets no further iteration
            else if (d0 <= 0.98 * tol2 * q.eta2) { q.done = 1; q.beta = q.gam = q.alpha = st_z(zero); }
        }
        break;
    case SC_RESTART:  // after r0 := r: rho = <r0, r> = ||r||^2 (the value SC_RHO / SC_TRUE left in r2)
        if (q.restart) { q.rho = make_double2(q.r2, 0.); q.r0n2 = q.r2; q.beta = st_z(zero); q.restart = 0; }
        break;
    // ---- merged iteration (solver.cu): alpha is known before Mhat p, rho' comes from <r0,s> - omega <r0,t> ----
    case SC_OMEGA2: {  // (d0,d1) = <t,s>, d2 = <t,t>, (e0,e1) = <r0,t>, (e2,e3) = <r0,s>
        zs om = zero, be = zero, ga = zero;
        q.want_update = 0;
        q.claim = 0;
        if (q.restart == 2) q.restart = 1;  // the minimal-residual step after a breakdown is done: restart before the next iteration
        if (!q.done) {
            if (!isfinite(d2) || !isfinite(d0) || !isfinite(d1) || !isfinite(e0) || !isfinite(e1) || !isfinite(e2) || !isfinite(e3)) {
                q.done = 1; q.status = 3; q.alpha = st_z(zero);
            } else {
                if (d2 > 0.) om = zs{d0 / d2, d1 / d2};
                const zs rho = ld_z(q.rho), rho1{e2 - (om.re * e0 - om.im * e1), e3 - (om.re * e1 + om.im * e0)};
                const double om2 = om.re * om.re + om.im * om.im, rh2 = rho.re * rho.re + rho.im * rho.im;
                if (!(om2 > 0.) || !(rh2 > 0.)) q.want_update = 1;  // stagnation: let the fp64 residual decide, beta = 0 gives p = r
                else {
                    ga = zdiv(rho1, rho);
                    be = zmul(ga, zdiv(ld_z(q.alpha), om));
                }
                if (!finite_z(be) || !finite_z(ga) || q.restart) be = ga = zero;
                q.rho = st_z(rho1);
            }
        }
        q.omega = st_z(om);
        q.beta = st_z(be);
        q.gam = st_z(ga);
        break;
    }
    case SC_RHO2: {  // (d0,d1) = <q0, p_new> = <r0, Mhat p_new>, d2 = ||r||^2
        zs al = zero;
        if (!q.done) {
            q.r2 = d2;
            if (d2 > q.maxr2) q.maxr2 = d2;
            if (!isfinite(d2) || !isfinite(d0) || !isfinite(d1)) { q.done = 1; q.status = 3; }
            else {
                if (d2 < q.delta2 * q.maxr2 || ++q.since >= leg_max) q.want_update = 1;
                q.claim = (d2 <= tol2 * q.eta2) ? 1 : 0;
                {   // relative breakdown (as in the oracle): rho' = <r0, r'> (left in q.rho by SC_OMEGA2) is noise against ||r0|| ||r'||
                    const zs rho = ld_z(q.rho);
                    if (d2 > 0. && !q.restart && !q.claim && rho.re * rho.re + rho.im * rho.im <= brk2 * q.r0n2 * d2 && q.nrestart < MAX_RESTARTS) {
                        q.restart = 1;   // r0 := p := r, q0 := Mhat^+ r0, rho := ||r||^2, alpha from SC_RESTART2 before the next iteration
                        q.nrestart++;
                    }
                }
                if (q.restart != 1) {  // (a restart recomputes alpha itself)
                    if (d0 * d0 + d1 * d1 > 0.) al = zdiv(ld_z(q.rho), zs{d0, d1});
                    if (!(d0 * d0 + d1 * d1 > 0.) || !finite_z(al)) {
                        // breakdown: the next iteration is a pure minimal-residual step (alpha = 0), then r0 := r (R11)
                        al = zero;
                        if (q.nrestart < MAX_RESTARTS) { q.restart = 2; q.nrestart++; }
                        else { q.done = 1; q.status = 2; }
                    }
                }
            }
        }
        q.alpha = st_z(al);
        break;
    }
    case SC_RESTART2:  // after r0 := p := r, q0 := Mhat^+ r0 for the flagged rhs: (d0,d1) = <q0, p>; rho = ||r||^2 (left in r2)
        if (q.restart == 1) {
            zs al = zero;
            q.restart = 0;
            q.rho = make_double2(q.r2, 0.);
            q.r0n2 = q.r2;
            q.beta = q.gam = st_z(zero);
            if (!q.done) {
                if (d0 * d0 + d1 * d1 > 0.) al = zdiv(ld_z(q.rho), zs{d0, d1});
                if (!(d0 * d0 + d1 * d1 > 0.) || !finite_z(al)) { al = zero; q.done = 1; q.status = isfinite(d0) && isfinite(d1) ? 2 : 3; }
            }
            q.alpha = st_z(al);
        }
        break;
    case SC_CONFIRM:  // d0 + d1 = ||eta - D psi||^2 on the full lattice, computed because every active rhs claimed convergence
        q.claim = 0;
        if (!q.done) {
            const double f = d0 + d1;
            if (!isfinite(f)) { q.done = 1; q.status = 3; }
            else if (f <= tol2 * q.eta2) { q.done = 1; q.true_r2 = f; q.alpha = q.beta = q.gam = st_z(zero); }
        }
        if (q.done) q.r2 = d0 + d1;  // (a rhs that failed keeps its iterated ||r||^2; the reliable update that follows replaces it)
        break;
    case SC_FINAL:  // d0 + d1 = ||eta - D psi||^2 on the full lattice; stored in r2 (true_r2 keeps the even-odd value)
        q.r2 = d0 + d1;
        break;
    }
    if (publish) {  // flag read-back without another launch: this rhs' scalars go straight into mapped pinned host memory
        static_assert(sizeof(RhsScalars) % 8 == 0, "RhsScalars is copied in 8-byte words");
        const unsigned long long *src = reinterpret_cast<const unsigned long long *>(&q);
        volatile unsigned long long *dst = reinterpret_cast<volatile unsigned long long *>(publish + rhs);
        for (int w = 0; w < (int)(sizeof(RhsScalars) / 8); w++) dst[w] = src[w];
        __threadfence_system();
    }
}

// ---- host wrappers ---------------------------------------------------------------------------------------
#define BLAS_LAUNCHED(c) do { if ((c).launches) ++*(c).launches; } while (0)

template <typename R> int blas_s_update(const BlasCtx &c, const typename Vec<R>::T *r, const typename Vec<R>::T *v, typename Vec<R>::T *s)
{
    const size_t n = field_vecs<R>(*c.g, c.B);
    s_update_kernel<<<blas_grid(n), BLAS_BLOCK, 0, c.st>>>(n, c.B, c.sc, r, v, s);
    BLAS_LAUNCHED(c);
    CLV_CUDA(cudaGetLastError());
    return 0;
}
template <typename R>
int blas_xr_update(const BlasCtx &c, typename Vec<R>::T *x, typename Vec<R>::T *r, const typename Vec<R>::T *p, const typename Vec<R>::T *s,
                   const typename Vec<R>::T *t, const typename Vec<R>::T *r0, int *nblocks)
{
    const size_t n = field_vecs<R>(*c.g, c.B);
    const int grid = blas_grid(n);
    xr_update_kernel<<<grid, BLAS_BLOCK, 0, c.st>>>(n, c.B, c.sc, x, r, p, s, t, r0, c.partial);
    BLAS_LAUNCHED(c);
    *nblocks = grid;
    CLV_CUDA(cudaGetLastError());
    return 0;
}
template <typename R> int blas_p_update(const BlasCtx &c, typename Vec<R>::T *p, const typename Vec<R>::T *r, const typename Vec<R>::T *v)
{
    const size_t n = field_vecs<R>(*c.g, c.B);
    p_update_kernel<<<blas_grid(n), BLAS_BLOCK, 0, c.st>>>(n, c.B, c.sc, p, r, v);
    BLAS_LAUNCHED(c);
    CLV_CUDA(cudaGetLastError());
    return 0;
}
template <typename R> int blas_restart(const BlasCtx &c, const typename Vec<R>::T *r, typename Vec<R>::T *r0, typename Vec<R>::T *p)
{
    const size_t n = field_vecs<R>(*c.g, c.B);
    restart_kernel<<<blas_grid(n), BLAS_BLOCK, 0, c.st>>>(n, c.B, c.sc, r, r0, p);
    BLAS_LAUNCHED(c);
    CLV_CUDA(cudaGetLastError());
    return 0;
}
template <typename R>
int blas_xrp_update(const BlasCtx &c, typename Vec<R>::T *x, typename Vec<R>::T *r, typename Vec<R>::T *p, const typename Vec<R>::T *s,
                    const typename Vec<R>::T *t, const typename Vec<R>::T *q0, int *nblocks)
{
    const size_t n = field_vecs<R>(*c.g, c.B);
    const int grid = blas_grid(n);
    xrp_update_kernel<<<grid, BLAS_BLOCK, 0, c.st>>>(n, c.B, c.sc, x, r, p, s, t, q0, c.partial);
    BLAS_LAUNCHED(c);
    *nblocks = grid;
    CLV_CUDA(cudaGetLastError());
    return 0;
}
template <typename R> int blas_gamma5(const BlasCtx &c, const typename Vec<R>::T *in, typename Vec<R>::T *out, int masked)
{
    const size_t n = field_vecs<R>(*c.g, c.B);
    gamma5_kernel<typename Vec<R>::T, Vec<R>::NV><<<blas_grid(n), BLAS_BLOCK, 0, c.st>>>(n, c.B, c.sc, masked, in, out);
    BLAS_LAUNCHED(c);
    CLV_CUDA(cudaGetLastError());
    return 0;
}
template <typename R> int blas_cdot(const BlasCtx &c, const typename Vec<R>::T *a, const typename Vec<R>::T *b, int *nblocks)
{
    const size_t n = field_vecs<R>(*c.g, c.B);
    const int grid = blas_grid(n);
    cdot_kernel<<<grid, BLAS_BLOCK, 0, c.st>>>(n, c.B, a, b, c.partial);
    BLAS_LAUNCHED(c);
    *nblocks = grid;
    CLV_CUDA(cudaGetLastError());
    return 0;
}
template <typename R> int blas_accumulate_y(const BlasCtx &c, double2 *y, typename Vec<R>::T *x)
{
    const size_t n = field_vecs<R>(*c.g, c.B);
    accumulate_y_kernel<<<blas_grid(n), BLAS_BLOCK, 0, c.st>>>(n, y, x);
    BLAS_LAUNCHED(c);
    CLV_CUDA(cudaGetLastError());
    return 0;
}
template <typename R> int blas_residual(const BlasCtx &c, const double2 *b, const double2 *w, double2 *r64, typename Vec<R>::T *rs, int *nblocks)
{
    const size_t n = field_vecs<double>(*c.g, c.B);
    const int grid = blas_grid(n);
    residual_kernel<<<grid, BLAS_BLOCK, 0, c.st>>>(n, c.B, b, w, r64, rs, c.partial);
    BLAS_LAUNCHED(c);
    *nblocks = grid;
    CLV_CUDA(cudaGetLastError());
    return 0;
}
int blas_norm2_pair(const BlasCtx &c, const double2 *a1, const double2 *b1, const double2 *a2, const double2 *b2, int *nblocks)
{
    const size_t n = field_vecs<double>(*c.g, c.B);
    const int grid = blas_grid(n);
    norm2_pair_kernel<<<grid, BLAS_BLOCK, 0, c.st>>>(n, c.B, a1, b1, a2, b2, c.partial);
    BLAS_LAUNCHED(c);
    *nblocks = grid;
    CLV_CUDA(cudaGetLastError());
    return 0;
}
int blas_scalar_step(const BlasCtx &c, int step, int nblocks, double tol2, double delta2, RhsScalars *publish)
{
    static const int leg_max = [] { const char *e = getenv("CLOVER_LEGMAX"); const int n = e ? atoi(e) : 0; return n > 0 ? n : LEG_MAX; }();  // tuning/debug knob only
    scalar_kernel<<<dim3(c.B, SC_SLICES), 256, 0, c.st>>>(step, c.B, nblocks, c.partial, step == SC_OMEGA2 ? c.partial2 : nullptr, c.sc, tol2, delta2, c.stage,
                                                          c.ticket, publish, leg_max, c.brk2);
    BLAS_LAUNCHED(c);
    CLV_CUDA(cudaGetLastError());
    return 0;
}

#define INST(R)                                                                                                                                  \
    template int blas_s_update<R>(const BlasCtx &, const Vec<R>::T *, const Vec<R>::T *, Vec<R>::T *);                                           \
    template int blas_xr_update<R>(const BlasCtx &, Vec<R>::T *, Vec<R>::T *, const Vec<R>::T *, const Vec<R>::T *, const Vec<R>::T *,          \
                                   const Vec<R>::T *, int *);                                                                                    \
    template int blas_p_update<R>(const BlasCtx &, Vec<R>::T *, const Vec<R>::T *, const Vec<R>::T *);                                           \
    template int blas_restart<R>(const BlasCtx &, const Vec<R>::T *, Vec<R>::T *, Vec<R>::T *);                                                                \
    template int blas_xrp_update<R>(const BlasCtx &, Vec<R>::T *, Vec<R>::T *, Vec<R>::T *, const Vec<R>::T *, const Vec<R>::T *,                   \
                                    const Vec<R>::T *, int *);                                                                                   \
    template int blas_gamma5<R>(const BlasCtx &, const Vec<R>::T *, Vec<R>::T *, int);                                                           \
    template int blas_cdot<R>(const BlasCtx &, const Vec<R>::T *, const Vec<R>::T *, int *);                                                     \
    template int blas_accumulate_y<R>(const BlasCtx &, double2 *, Vec<R>::T *);                                                                  \
    template int blas_residual<R>(const BlasCtx &, const double2 *, const double2 *, double2 *, Vec<R>::T *, int *);
INST(float)
INST(double)
#undef INST

}  // namespace clv
