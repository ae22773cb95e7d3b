// setup.cu -- one-time kernels of clover_create and the canonical <-> internal reorders
// (the paper's "reordering of the arrays between the two libraries").
#include "context.h"
#include <cstdarg>
#include <cstdio>

namespace clv {

typedef cx<double> zc;

struct Lex {
    int x[4];
};
__device__ __forceinline__ long lex_index(const Geom &g, const Lex &c)
{
    return (((long)c.x[3] * g.Z + c.x[2]) * g.Y + c.x[1]) * g.X + c.x[0];
}
__device__ __forceinline__ Lex lex_of(const Geom &g, int cb, int p)
{
    Coord c = decode(g, cb, p);
    Lex l;
    l.x[0] = c.x; l.x[1] = c.y; l.x[2] = c.z; l.x[3] = c.t;
    return l;
}
__device__ __forceinline__ Lex shifted(const Geom &g, Lex c, int mu, int step)
{
    const int n = (mu == 0) ? g.X : (mu == 1) ? g.Y : (mu == 2) ? g.Z : g.T;
    c.x[mu] = (c.x[mu] + step + n) % n;
    return c;
}
__device__ __forceinline__ void ld_link(const double *__restrict__ gauge, long V, int mu, long lex, zc u[9])
{
    const double2 *p = reinterpret_cast<const double2 *>(gauge) + ((long)mu * V + lex) * 9;
#pragma unroll
    for (int k = 0; k < 9; k++) {
        double2 v = __ldg(p + k);
        u[k] = mk<double>(v.x, v.y);
    }
}

// ---- S0: links canonical -> internal (fp64 full, fp32 full or two-row) --------------------------
template <int RECON32>
__global__ void reorder_gauge_kernel(Geom g, const double *__restrict__ gauge, OpData<double> o64, OpData<float> o32)
{
    const int cb = blockIdx.x * blockDim.x + threadIdx.x;
    if (cb >= g.Vh) return;
    const int p = blockIdx.y >> 2, mu = blockIdx.y & 3;
    const long V = 2L * g.Vh;
    zc u[9];
    ld_link(gauge, V, mu, lex_index(g, lex_of(g, cb, p)), u);
#pragma unroll
    for (int k = 0; k < 9; k++) o64.gauge[p][mu][lb_index(cb, k, 9)] = make_double2(u[k].re, u[k].im);
#pragma unroll
    for (int k = 0; k < RECON32 / 2; k++) o32.gauge[p][mu][cplx_index<float>(cb, k, RECON32 / 2)] = make_float2((float)u[k].re, (float)u[k].im);
}

// Site-major copies for the B = 8 kernels: per output site of parity p the 8 links of its hop, in the order d = 2 mu + (fwd ? 0 : 1)
// (fwd: U_mu(x); bwd: U_mu(x - mu), stored as it is and daggered in-kernel); fp32 rounded exactly as the lane-blocked copy is.
template <typename R, int RECON> __global__ void pack_links_kernel(Geom g, const double *__restrict__ gauge, OpData<R> o)
{
    const int cb = blockIdx.x * blockDim.x + threadIdx.x;
    if (cb >= g.Vh) return;
    const int p = blockIdx.y >> 3, d = blockIdx.y & 7, mu = d >> 1;
    const long V = 2L * g.Vh;
    const Lex x = lex_of(g, cb, p);
    zc u[9];
    ld_link(gauge, V, mu, lex_index(g, (d & 1) ? shifted(g, x, mu, -1) : x), u);
    R *dst = o.pk_link[p] + (size_t)cb * pk_link_stride(RECON) + d * RECON;
#pragma unroll
    for (int k = 0; k < RECON / 2; k++) {
        dst[2 * k] = (R)u[k].re;
        dst[2 * k + 1] = (R)u[k].im;
    }
}
// lane-blocked packed clover blocks (36 complex per site) -> 72 consecutive reals per site
template <typename R> __global__ void pack_clover_kernel(Geom g, OpData<R> o)
{
    const unsigned i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= (unsigned)g.Vh * 36u) return;
    const unsigned cb = i / 36u, k = i % 36u;
    const int p = blockIdx.y >> 1;
    const typename Vec<R>::C *src = (blockIdx.y & 1) ? o.clov_inv[p] : o.clov[p];
    R *dst = ((blockIdx.y & 1) ? o.pk_clov_inv[p] : o.pk_clov[p]) + (size_t)cb * PK_CLOV_STRIDE + 2 * k;
    const typename Vec<R>::C v = src[cplx_index<R>(cb, k, 36)];
    dst[0] = v.x;
    dst[1] = v.y;
}

// ---- S1: clover term ------------------------------------------------------------------------------
__device__ __forceinline__ void mm(const zc a[9], const zc b[9], zc c[9])  // c = a b
{
#pragma unroll
    for (int i = 0; i < 3; i++)
#pragma unroll
        for (int j = 0; j < 3; j++) {
            zc s = mk<double>(0, 0);
#pragma unroll
            for (int k = 0; k < 3; k++) fma_cx(s, a[i * 3 + k], b[k * 3 + j]);
            c[i * 3 + j] = s;
        }
}
__device__ __forceinline__ void mmd(const zc a[9], const zc b[9], zc c[9])  // c = a b^dagger
{
#pragma unroll
    for (int i = 0; i < 3; i++)
#pragma unroll
        for (int j = 0; j < 3; j++) {
            zc s = mk<double>(0, 0);
#pragma unroll
            for (int k = 0; k < 3; k++) fma_cx(s, a[i * 3 + k], conj(b[j * 3 + k]));
            c[i * 3 + j] = s;
        }
}
__device__ __forceinline__ void mdm(const zc a[9], const zc b[9], zc c[9])  // c = a^dagger b
{
#pragma unroll
    for (int i = 0; i < 3; i++)
#pragma unroll
        for (int j = 0; j < 3; j++) {
            zc s = mk<double>(0, 0);
#pragma unroll
            for (int k = 0; k < 3; k++) fma_conj(s, a[k * 3 + i], b[k * 3 + j]);
            c[i * 3 + j] = s;
        }
}

__device__ __forceinline__ void mdmd(const zc a[9], const zc b[9], zc c[9])  // c = a^dagger b^dagger
{
#pragma unroll
    for (int i = 0; i < 3; i++)
#pragma unroll
        for (int j = 0; j < 3; j++) {
            zc s = mk<double>(0, 0);
#pragma unroll
            for (int k = 0; k < 3; k++) fma_cx(s, conj(a[k * 3 + i]), conj(b[j * 3 + k]));
            c[i * 3 + j] = s;
        }
}

// Fhat_{mu nu}(x) = (Q - Q^dagger)/8, Q = sum of the four leaves based at x
__device__ void fhat_plane(const Geom &g, const double *__restrict__ gauge, const Lex &x, int mu, int nu, zc F[9])
{
    const long V = 2L * g.Vh;
    const Lex xpm = shifted(g, x, mu, +1), xpn = shifted(g, x, nu, +1);
    const Lex xmm = shifted(g, x, mu, -1), xmn = shifted(g, x, nu, -1);
    const Lex xmmpn = shifted(g, xmm, nu, +1), xmmmn = shifted(g, xmm, nu, -1), xpmmn = shifted(g, xpm, nu, -1);
    zc a[9], b[9], c[9], d[9], t1[9], t2[9], Q[9];
    // L1 = U_mu(x) U_nu(x+mu) U_mu(x+nu)^+ U_nu(x)^+
    ld_link(gauge, V, mu, lex_index(g, x), a);
    ld_link(gauge, V, nu, lex_index(g, xpm), b);
    ld_link(gauge, V, mu, lex_index(g, xpn), c);
    ld_link(gauge, V, nu, lex_index(g, x), d);
    mm(a, b, t1); mmd(t1, c, t2); mmd(t2, d, Q);
    // L2 = U_nu(x) U_mu(x-mu+nu)^+ U_nu(x-mu)^+ U_mu(x-mu)
    ld_link(gauge, V, mu, lex_index(g, xmmpn), b);
    ld_link(gauge, V, nu, lex_index(g, xmm), c);
    ld_link(gauge, V, mu, lex_index(g, xmm), a);
    mmd(d, b, t1); mmd(t1, c, t2); mm(t2, a, t1);
#pragma unroll
    for (int i = 0; i < 9; i++) Q[i] = Q[i] + t1[i];
    // L3 = U_mu(x-mu)^+ U_nu(x-mu-nu)^+ U_mu(x-mu-nu) U_nu(x-nu)
    ld_link(gauge, V, nu, lex_index(g, xmmmn), b);
    ld_link(gauge, V, mu, lex_index(g, xmmmn), c);
    ld_link(gauge, V, nu, lex_index(g, xmn), d);
    mdmd(a, b, t1);
    mm(t1, c, t2); mm(t2, d, t1);
#pragma unroll
    for (int i = 0; i < 9; i++) Q[i] = Q[i] + t1[i];
    // L4 = U_nu(x-nu)^+ U_mu(x-nu) U_nu(x+mu-nu) U_mu(x)^+
    ld_link(gauge, V, mu, lex_index(g, xmn), b);
    ld_link(gauge, V, nu, lex_index(g, xpmmn), c);
    ld_link(gauge, V, mu, lex_index(g, x), a);
    mdm(d, b, t1); mm(t1, c, t2); mmd(t2, a, t1);
#pragma unroll
    for (int i = 0; i < 9; i++) Q[i] = Q[i] + t1[i];
#pragma unroll
    for (int i = 0; i < 3; i++)
#pragma unroll
        for (int j = 0; j < 3; j++) F[i * 3 + j] = 0.125 * (Q[i * 3 + j] - conj(Q[j * 3 + i]));
}

// in-place inverse of a 6x6 complex matrix, Gauss-Jordan with partial pivoting; returns false if singular
__device__ bool invert6(zc M[6][6])
{
    zc W[6][6];
    for (int i = 0; i < 6; i++)
        for (int j = 0; j < 6; j++) W[i][j] = mk<double>(i == j ? 1.0 : 0.0, 0.0);
    for (int col = 0; col < 6; col++) {
        int piv = col;
        double best = M[col][col].re * M[col][col].re + M[col][col].im * M[col][col].im;
        for (int r = col + 1; r < 6; r++) {
            double m = M[r][col].re * M[r][col].re + M[r][col].im * M[r][col].im;
            if (m > best) { best = m; piv = r; }
        }
        if (!(best > 0.0)) return false;
        if (piv != col)
            for (int j = 0; j < 6; j++) {
                zc t = M[col][j]; M[col][j] = M[piv][j]; M[piv][j] = t;
                t = W[col][j]; W[col][j] = W[piv][j]; W[piv][j] = t;
            }
        const zc d = (1.0 / best) * conj(M[col][col]);
        for (int j = 0; j < 6; j++) { M[col][j] = d * M[col][j]; W[col][j] = d * W[col][j]; }
        for (int r = 0; r < 6; r++) {
            if (r == col) continue;
            const zc f = M[r][col];
            for (int j = 0; j < 6; j++) {
                M[r][j] = M[r][j] - f * M[col][j];
                W[r][j] = W[r][j] - f * W[col][j];
            }
        }
    }
    for (int i = 0; i < 6; i++)
        for (int j = 0; j < 6; j++) M[i][j] = W[i][j];
    return true;
}

// pack a Hermitian 6x6 block: 3 complex holding the 6 real diagonals, then the 15 lower off-diagonals row by row
__device__ void pack_block(const zc M[6][6], int blk, unsigned cb, double2 *o64, float2 *o32)
{
    for (int k = 0; k < 3; k++) {
        const double a = M[2 * k][2 * k].re, b = M[2 * k + 1][2 * k + 1].re;
        o64[lb_index(cb, 18 * blk + k, 36)] = make_double2(a, b);
        o32[cplx_index<float>(cb, 18 * blk + k, 36)] = make_float2((float)a, (float)b);
    }
    int k = 3;
    for (int i = 1; i < 6; i++)
        for (int j = 0; j < i; j++, k++) {
            // Hermitian average of the two triangles (they agree to rounding)
            const double re = 0.5 * (M[i][j].re + M[j][i].re), im = 0.5 * (M[i][j].im - M[j][i].im);
            o64[lb_index(cb, 18 * blk + k, 36)] = make_double2(re, im);
            o32[cplx_index<float>(cb, 18 * blk + k, 36)] = make_float2((float)re, (float)im);
        }
}

__global__ void clover_build_kernel(Geom g, const double *__restrict__ gauge, double csw_kappa, OpData<double> o64, OpData<float> o32,
                                    int *singular)
{
    const int cb = blockIdx.x * blockDim.x + threadIdx.x;
    if (cb >= g.Vh) return;
    const int p = blockIdx.y;
    const Lex x = lex_of(g, cb, p);
    zc F01[9], F02[9], F03[9], F12[9], F13[9], F23[9];
    fhat_plane(g, gauge, x, 0, 1, F01);
    fhat_plane(g, gauge, x, 0, 2, F02);
    fhat_plane(g, gauge, x, 0, 3, F03);
    fhat_plane(g, gauge, x, 1, 2, F12);
    fhat_plane(g, gauge, x, 1, 3, F13);
    fhat_plane(g, gauge, x, 2, 3, F23);
    for (int blk = 0; blk < 2; blk++) {
        const double sg = blk ? -1.0 : 1.0;
        zc M[6][6];
        // block = 1 + i c [ sigma1 (x) E1 + sigma2 (x) E2 + sigma3 (x) E3 ],
        // E1 = sg F03 - F12, E2 = sg F13 + F02, E3 = sg F23 - F01   (chiral basis)
        for (int a = 0; a < 3; a++)
            for (int b = 0; b < 3; b++) {
                const int i = a * 3 + b;
                const zc E1 = sg * F03[i] - F12[i], E2 = sg * F13[i] + F02[i], E3 = sg * F23[i] - F01[i];
                const zc iE3 = mk<double>(-E3.im, E3.re);
                const zc lo = add_i(E1, E2);  // E1 + i E2  (row spin 1, col spin 0)
                const zc up = sub_i(E1, E2);  // E1 - i E2  (row spin 0, col spin 1)
                const double dl = (a == b) ? 1.0 : 0.0;
                M[a][b] = mk<double>(dl + csw_kappa * iE3.re, csw_kappa * iE3.im);
                M[3 + a][3 + b] = mk<double>(dl - csw_kappa * iE3.re, -csw_kappa * iE3.im);
                M[a][3 + b] = mk<double>(-csw_kappa * up.im, csw_kappa * up.re);
                M[3 + a][b] = mk<double>(-csw_kappa * lo.im, csw_kappa * lo.re);
            }
        pack_block(M, blk, cb, o64.clov[p], o32.clov[p]);
        if (!invert6(M)) atomicAdd(singular, 1);
        pack_block(M, blk, cb, o64.clov_inv[p], o32.clov_inv[p]);
    }
}

// ---- canonical <-> internal spinor reorders ------------------------------------------------------
template <typename CT> struct CanonC;
template <> struct CanonC<double> { typedef double2 T; };
template <> struct CanonC<float> { typedef float2 T; };

// One CTA of 384 threads moves one 32-lane block of j = cb*B + rhs (x 12 complex) through shared memory, so that both sides
// are coalesced: the canonical side in 192-byte chunks (one (site, rhs) spinor each), the internal side in 512-byte rows.
constexpr int RO_THREADS = 384;

template <typename CT, typename R> __global__ void __launch_bounds__(RO_THREADS) reorder_in_kernel(Geom g, const CT *__restrict__ canon, typename Vec<R>::T *even,
                                                                                                  typename Vec<R>::T *odd, int B)
{
    __shared__ double2 sm[12][33];
    const int p = blockIdx.y;
    const long V = 2L * g.Vh;
    {
        const int chunk = threadIdx.x / 12, k = threadIdx.x % 12;
        const unsigned j = blockIdx.x * 32u + chunk;
        double2 v = make_double2(0., 0.);
        if (j < (unsigned)g.Vh * B) {
            const int cb = j / B, rhs = j % B;
            const typename CanonC<CT>::T e = __ldg(reinterpret_cast<const typename CanonC<CT>::T *>(canon) + ((long)rhs * V + lex_index(g, lex_of(g, cb, p))) * 12 + k);
            v = make_double2((double)e.x, (double)e.y);
        }
        sm[k][chunk] = v;
    }
    __syncthreads();
    typename Vec<R>::T *f = p ? odd : even;
    const int lane = threadIdx.x & 31, row = threadIdx.x >> 5;   // 12 rows of 32 lanes
    if (sizeof(R) == 8) {
        reinterpret_cast<double2 *>(f)[((size_t)blockIdx.x * 12 + row) * 32 + lane] = sm[row][lane];
    } else if (row < 6) {
        const double2 a = sm[2 * row][lane], b = sm[2 * row + 1][lane];
        reinterpret_cast<float4 *>(f)[((size_t)blockIdx.x * 6 + row) * 32 + lane] = make_float4((float)a.x, (float)a.y, (float)b.x, (float)b.y);
    }
}

template <typename CT, typename R> __global__ void __launch_bounds__(RO_THREADS) reorder_out_kernel(Geom g, CT *canon, const typename Vec<R>::T *__restrict__ even,
                                                                                                   const typename Vec<R>::T *__restrict__ odd, int B)
{
    __shared__ double2 sm[12][33];
    const int p = blockIdx.y;
    const long V = 2L * g.Vh;
    const typename Vec<R>::T *f = p ? odd : even;
    {
        const int lane = threadIdx.x & 31, row = threadIdx.x >> 5;
        if (!f) sm[row][lane] = make_double2(0., 0.);
        else if (sizeof(R) == 8) sm[row][lane] = __ldg(reinterpret_cast<const double2 *>(f) + ((size_t)blockIdx.x * 12 + row) * 32 + lane);
        else if (row < 6) {
            const float4 v = __ldg(reinterpret_cast<const float4 *>(f) + ((size_t)blockIdx.x * 6 + row) * 32 + lane);
            sm[2 * row][lane] = make_double2((double)v.x, (double)v.y);
            sm[2 * row + 1][lane] = make_double2((double)v.z, (double)v.w);
        }
    }
    __syncthreads();
    const int chunk = threadIdx.x / 12, k = threadIdx.x % 12;
    const unsigned j = blockIdx.x * 32u + chunk;
    if (j >= (unsigned)g.Vh * B) return;
    const int cb = j / B, rhs = j % B;
    const double2 v = sm[k][chunk];
    typename CanonC<CT>::T e;
    e.x = (CT)v.x;
    e.y = (CT)v.y;
    reinterpret_cast<typename CanonC<CT>::T *>(canon)[((long)rhs * V + lex_index(g, lex_of(g, cb, p))) * 12 + k] = e;
}

template <typename CT, typename R>
int reorder_in(const Geom &g, const CT *canon, typename Vec<R>::T *even, typename Vec<R>::T *odd, int B, cudaStream_t st)
{
    dim3 grid(lb_blocks((unsigned)g.Vh * B), 2);
    reorder_in_kernel<CT, R><<<grid, RO_THREADS, 0, st>>>(g, canon, even, odd, B);
    CLV_CUDA(cudaGetLastError());
    return 0;
}
// a null even/odd pointer writes zeros to that parity
template <typename CT, typename R>
int reorder_out(const Geom &g, CT *canon, const typename Vec<R>::T *even, const typename Vec<R>::T *odd, int B, cudaStream_t st)
{
    dim3 grid(lb_blocks((unsigned)g.Vh * B), 2);
    reorder_out_kernel<CT, R><<<grid, RO_THREADS, 0, st>>>(g, canon, even, odd, B);
    CLV_CUDA(cudaGetLastError());
    return 0;
}
template int reorder_in<double, double>(const Geom &, const double *, double2 *, double2 *, int, cudaStream_t);
template int reorder_in<float, float>(const Geom &, const float *, float4 *, float4 *, int, cudaStream_t);
template int reorder_out<double, double>(const Geom &, double *, const double2 *, const double2 *, int, cudaStream_t);
template int reorder_out<float, float>(const Geom &, float *, const float4 *, const float4 *, int, cudaStream_t);

// ---- clover_create's device work ---------------------------------------------------------------
template <typename T> static int dev_alloc(clover_ctx *ctx, T **p, size_t count, cudaStream_t st)
{
    void *q = nullptr;
    CLV_CUDA(cudaMalloc(&q, count * sizeof(T)));
    ctx->allocs.push_back(q);
    CLV_CUDA(cudaMemsetAsync(q, 0, count * sizeof(T), st));   // padding lanes must read as zeros; ordered before the fill kernels on `st`
    *p = (T *)q;
    return 0;
}

int setup_operator(clover_ctx *ctx, const double *gauge_dev, cudaStream_t st)
{
    const Geom &g = ctx->geom;
    const size_t nb = lb_blocks(g.Vh) * 32u;  // padded entries per parity
    for (int p = 0; p < 2; p++) {
        for (int mu = 0; mu < 4; mu++) {
            CLV_CHECK(dev_alloc(ctx, &ctx->op64.gauge[p][mu], nb * 9, st));
            CLV_CHECK(dev_alloc(ctx, &ctx->op32.gauge[p][mu], nb * (ctx->op32.recon / 2), st));
        }
        CLV_CHECK(dev_alloc(ctx, &ctx->op64.clov[p], nb * 36, st));
        CLV_CHECK(dev_alloc(ctx, &ctx->op64.clov_inv[p], nb * 36, st));
        CLV_CHECK(dev_alloc(ctx, &ctx->op32.clov[p], nb * 36, st));
        CLV_CHECK(dev_alloc(ctx, &ctx->op32.clov_inv[p], nb * 36, st));
    }
    for (int p = 0; p < 2; p++) {
        CLV_CHECK(dev_alloc(ctx, &ctx->op64.pk_link[p], (size_t)g.Vh * pk_link_stride(18), st));
        CLV_CHECK(dev_alloc(ctx, &ctx->op64.pk_clov[p], (size_t)g.Vh * PK_CLOV_STRIDE, st));
        CLV_CHECK(dev_alloc(ctx, &ctx->op64.pk_clov_inv[p], (size_t)g.Vh * PK_CLOV_STRIDE, st));
        CLV_CHECK(dev_alloc(ctx, &ctx->op32.pk_link[p], (size_t)g.Vh * pk_link_stride(ctx->op32.recon), st));
        CLV_CHECK(dev_alloc(ctx, &ctx->op32.pk_clov[p], (size_t)g.Vh * PK_CLOV_STRIDE, st));
        CLV_CHECK(dev_alloc(ctx, &ctx->op32.pk_clov_inv[p], (size_t)g.Vh * PK_CLOV_STRIDE, st));
    }
    CLV_CHECK(dev_alloc(ctx, &ctx->sched, 2, st));
    int *singular = nullptr;
    CLV_CHECK(dev_alloc(ctx, &singular, 1, st));
    dim3 gg((g.Vh + 127) / 128, 8);
    if (ctx->op32.recon == 12) reorder_gauge_kernel<12><<<gg, 128, 0, st>>>(g, gauge_dev, ctx->op64, ctx->op32);
    else reorder_gauge_kernel<18><<<gg, 128, 0, st>>>(g, gauge_dev, ctx->op64, ctx->op32);
    CLV_CUDA(cudaGetLastError());
    dim3 gc((g.Vh + 63) / 64, 2);
    clover_build_kernel<<<gc, 64, 0, st>>>(g, gauge_dev, ctx->csw * ctx->kappa, ctx->op64, ctx->op32, singular);
    CLV_CUDA(cudaGetLastError());
    dim3 gp((g.Vh + 127) / 128, 16);
    if (ctx->op32.recon == 12) pack_links_kernel<float, 12><<<gp, 128, 0, st>>>(g, gauge_dev, ctx->op32);
    else pack_links_kernel<float, 18><<<gp, 128, 0, st>>>(g, gauge_dev, ctx->op32);
    pack_links_kernel<double, 18><<<gp, 128, 0, st>>>(g, gauge_dev, ctx->op64);
    CLV_CUDA(cudaGetLastError());
    dim3 gk(((unsigned)g.Vh * 36u + 255u) / 256u, 4);
    pack_clover_kernel<float><<<gk, 256, 0, st>>>(g, ctx->op32);
    pack_clover_kernel<double><<<gk, 256, 0, st>>>(g, ctx->op64);
    CLV_CUDA(cudaGetLastError());
    int h = 0;
    CLV_CUDA(cudaMemcpyAsync(&h, singular, sizeof(int), cudaMemcpyDeviceToHost, st));
    CLV_CUDA(cudaStreamSynchronize(st));
    if (h) {
        set_error("clover term is singular at %d blocks", h);
        return CLOVER_EINVAL;
    }
    return 0;
}

// ---- thread-local error string ------------------------------------------------------------------
static thread_local char g_err[512] = "no error";
void set_error(const char *fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof g_err, fmt, ap);
    va_end(ap);
}
const char *last_error() { return g_err; }

}  // namespace clv
