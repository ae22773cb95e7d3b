// dslash_kernel.cuh -- the Wilson-clover stencil kernel, one thread per (site, rhs).
//
//   out = P ( X + coef * H_{p,1-p} in ),   P = 1 | A_pp^-1,   X = 0 | xin | A_pp xin
//   (H psi)(x) = sum_mu [ f (1 - gamma_mu) U_mu(x) psi(x+mu) + g (1 + gamma_mu) U_mu(x-mu)^+ psi(x-mu) ]
//
// Spin projection in the chiral basis gamma_mu = [[0, B_mu], [B_mu^+, 0]], B_k = -i sigma_k, B_t = 1:
// (1 -+ gamma_mu) has rank 2, so only the half spinor h = psi_up -+ B psi_low is multiplied by the link,
// and the lower two spin rows of the result are -+ B^+ (U h).
// Thread mapping: j = cb*B + rhs, rhs fastest: the B rhs-lanes of a site share (broadcast) every link and
// clover load, and their spinor loads fill B*16 contiguous bytes per vector (one 128-byte line at B = 8).
#pragma once
#include "context.h"

namespace clv {

#ifndef CLV_DSLASH_BLOCK
#define CLV_DSLASH_BLOCK 128
#endif
#ifndef CLV_DSLASH_MINB
#define CLV_DSLASH_MINB 4 // <= 128 registers: measured best (ptxas keeps more loads in flight than with no hint; profiles/r1_tuning.md)
#endif
constexpr int DSLASH_BLOCK = CLV_DSLASH_BLOCK;

template <typename R, int MU, int FWD> __device__ __forceinline__ void project(const cx<R> psi[12], cx<R> h[6])
{
#pragma unroll
    for (int a = 0; a < 3; a++) {
        const cx<R> p0 = psi[a], p1 = psi[3 + a], p2 = psi[6 + a], p3 = psi[9 + a];
        if (MU == 0) {
            h[a] = FWD ? add_i(p0, p3) : sub_i(p0, p3);
            h[3 + a] = FWD ? add_i(p1, p2) : sub_i(p1, p2);
        } else if (MU == 1) {
            h[a] = FWD ? p0 + p3 : p0 - p3;
            h[3 + a] = FWD ? p1 - p2 : p1 + p2;
        } else if (MU == 2) {
            h[a] = FWD ? add_i(p0, p2) : sub_i(p0, p2);
            h[3 + a] = FWD ? sub_i(p1, p3) : add_i(p1, p3);
        } else {
            h[a] = FWD ? p0 - p2 : p0 + p2;
            h[3 + a] = FWD ? p1 - p3 : p1 + p3;
        }
    }
}

// acc += (g, -+ B^+ g)
template <typename R, int MU, int FWD> __device__ __forceinline__ void reconstruct(const cx<R> g[6], cx<R> acc[12])
{
#pragma unroll
    for (int a = 0; a < 3; a++) {
        const cx<R> g0 = g[a], g1 = g[3 + a];
        acc[a] = acc[a] + g0;
        acc[3 + a] = acc[3 + a] + g1;
        if (MU == 0) {  // B^+ g = (i g1, i g0)
            acc[6 + a] = FWD ? sub_i(acc[6 + a], g1) : add_i(acc[6 + a], g1);
            acc[9 + a] = FWD ? sub_i(acc[9 + a], g0) : add_i(acc[9 + a], g0);
        } else if (MU == 1) {  // (g1, -g0)
            acc[6 + a] = FWD ? acc[6 + a] - g1 : acc[6 + a] + g1;
            acc[9 + a] = FWD ? acc[9 + a] + g0 : acc[9 + a] - g0;
        } else if (MU == 2) {  // (i g0, -i g1)
            acc[6 + a] = FWD ? sub_i(acc[6 + a], g0) : add_i(acc[6 + a], g0);
            acc[9 + a] = FWD ? add_i(acc[9 + a], g1) : sub_i(acc[9 + a], g1);
        } else {  // (g0, g1)
            acc[6 + a] = FWD ? acc[6 + a] - g0 : acc[6 + a] + g0;
            acc[9 + a] = FWD ? acc[9 + a] - g1 : acc[9 + a] + g1;
        }
    }
}

template <typename R, int B, int RECON, int MU, int FWD>
__device__ __forceinline__ void hop_dir(const Geom &g, const OpData<R> &op, const typename Vec<R>::T *__restrict__ in, int p, int cb,
                                        int rhs, const Coord &c, cx<R> acc[12])
{
    bool wrap;
    const int nb = neighbour<MU, FWD>(g, cb, c, wrap);
    cx<R> psi[12], h[6], u[9], gh[6];
    load_spinor(in, (unsigned)nb * B + rhs, psi);
    // (ternaries rather than op.gauge[p]: runtime indexing of a kernel parameter would force a local copy)
    if (FWD) load_link<R, RECON>(p ? op.gauge[1][MU] : op.gauge[0][MU], cb, u);
    else load_link<R, RECON>(p ? op.gauge[0][MU] : op.gauge[1][MU], nb, u);
    project<R, MU, FWD>(psi, h);
    if (wrap && g.bc[MU] < 0) {
#pragma unroll
        for (int i = 0; i < 6; i++) h[i] = mk<R>(-h[i].re, -h[i].im);
    }
#pragma unroll
    for (int s = 0; s < 2; s++)
#pragma unroll
        for (int a = 0; a < 3; a++) {
            cx<R> t = mk<R>(0, 0);
#pragma unroll
            for (int b = 0; b < 3; b++) {
                if (FWD) fma_cx(t, u[a * 3 + b], h[s * 3 + b]);
                else fma_conj(t, u[b * 3 + a], h[s * 3 + b]);
            }
            gh[s * 3 + a] = t;
        }
    reconstruct<R, MU, FWD>(gh, acc);
}

// y (+)= M x for the two packed 6x6 Hermitian blocks of one site
template <typename R, bool ACCUM>
__device__ __forceinline__ void clover_mul(const typename Vec<R>::C *__restrict__ clov, unsigned cb, const cx<R> x[12], cx<R> y[12])
{
    const typename Vec<R>::C *p = clov + lb_index(cb, 0, 36);
#pragma unroll
    for (int blk = 0; blk < 2; blk++) {
        const int o = 6 * blk;
#pragma unroll
        for (int k = 0; k < 3; k++) {
            const typename Vec<R>::C d = __ldg(p + 32 * (18 * blk + k));
            if (ACCUM) {
                y[o + 2 * k] = y[o + 2 * k] + d.x * x[o + 2 * k];
                y[o + 2 * k + 1] = y[o + 2 * k + 1] + d.y * x[o + 2 * k + 1];
            } else {
                y[o + 2 * k] = d.x * x[o + 2 * k];
                y[o + 2 * k + 1] = d.y * x[o + 2 * k + 1];
            }
        }
        int k = 3;
#pragma unroll
        for (int i = 1; i < 6; i++)
#pragma unroll
            for (int j = 0; j < i; j++, k++) {
                const typename Vec<R>::C v = __ldg(p + 32 * (18 * blk + k));
                const cx<R> L = mk<R>(v.x, v.y);
                fma_cx(y[o + i], L, x[o + j]);
                fma_conj(y[o + j], L, x[o + i]);
            }
    }
}

// per-rhs block reduction of up to 3 doubles; rhs = threadIdx.x % B. Result of block b, rhs r at partial[(b*B + r)*4 + c].
template <int B, int BLOCK> __device__ __forceinline__ void block_reduce_rhs(double v0, double v1, double v2, double *__restrict__ partial)
{
    __shared__ double sm[BLOCK / 32][B][3];
#pragma unroll
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
    if (threadIdx.x < B * 3) {
        const int r = threadIdx.x / 3, c = threadIdx.x % 3;
        double s = 0;
#pragma unroll
        for (int w = 0; w < BLOCK / 32; w++) s += sm[w][r][c];
        partial[((size_t)blockIdx.x * B + r) * 4 + c] = s;
    }
}

template <typename R, int B, int RECON, int XMODE, int PINV, int DOT>
__global__ void __launch_bounds__(DSLASH_BLOCK, CLV_DSLASH_MINB) dslash_kernel(const Geom g, const OpData<R> op, const DslashArgs<R> a)
{
    const unsigned j = blockIdx.x * DSLASH_BLOCK + threadIdx.x;
    const bool active = j < (unsigned)g.Vh * B;
    double d0 = 0, d1 = 0, d2 = 0;
    if (active) {
        const int cb = j / B, rhs = j % B, p = a.parity;
        const Coord c = decode(g, cb, p);
        cx<R> acc[12];
#pragma unroll
        for (int i = 0; i < 12; i++) acc[i] = mk<R>(0, 0);
        hop_dir<R, B, RECON, 0, 1>(g, op, a.in, p, cb, rhs, c, acc);
        hop_dir<R, B, RECON, 0, 0>(g, op, a.in, p, cb, rhs, c, acc);
        hop_dir<R, B, RECON, 1, 1>(g, op, a.in, p, cb, rhs, c, acc);
        hop_dir<R, B, RECON, 1, 0>(g, op, a.in, p, cb, rhs, c, acc);
        hop_dir<R, B, RECON, 2, 1>(g, op, a.in, p, cb, rhs, c, acc);
        hop_dir<R, B, RECON, 2, 0>(g, op, a.in, p, cb, rhs, c, acc);
        hop_dir<R, B, RECON, 3, 1>(g, op, a.in, p, cb, rhs, c, acc);
        hop_dir<R, B, RECON, 3, 0>(g, op, a.in, p, cb, rhs, c, acc);
#pragma unroll
        for (int i = 0; i < 12; i++) acc[i] = a.coef * acc[i];
        cx<R> x[12];
        if (XMODE != XM_NONE) load_spinor(a.xin, j, x);
        if (XMODE == XM_PLAIN) {
#pragma unroll
            for (int i = 0; i < 12; i++) acc[i] = acc[i] + x[i];
        }
        if (XMODE == XM_CLOVER) clover_mul<R, true>(p ? op.clov[1] : op.clov[0], cb, x, acc);
        if (PINV) {
            cx<R> t[12];
            clover_mul<R, false>(p ? op.clov_inv[1] : op.clov_inv[0], cb, acc, t);
#pragma unroll
            for (int i = 0; i < 12; i++) acc[i] = t[i];
        }
        store_spinor(a.out, j, acc);
        if (DOT == DOT_W) {
            cx<R> w[12];
            load_spinor(a.w, j, w);
#pragma unroll
            for (int i = 0; i < 12; i++) {  // <w, out> = sum conj(w) out
                d0 += (double)(w[i].re * acc[i].re + w[i].im * acc[i].im);
                d1 += (double)(w[i].re * acc[i].im - w[i].im * acc[i].re);
            }
        }
        if (DOT == DOT_X) {
#pragma unroll
            for (int i = 0; i < 12; i++) {  // <out, xin> and <out, out>
                d0 += (double)(acc[i].re * x[i].re + acc[i].im * x[i].im);
                d1 += (double)(acc[i].re * x[i].im - acc[i].im * x[i].re);
                d2 += (double)(acc[i].re * acc[i].re + acc[i].im * acc[i].im);
            }
        }
    }
    if (DOT != DOT_NONE) block_reduce_rhs<B, DSLASH_BLOCK>(d0, d1, d2, a.partial);
}

// standalone clover apply: out = A in or A^-1 in
template <typename R, int B>
__global__ void __launch_bounds__(DSLASH_BLOCK) clover_kernel(const Geom g, const typename Vec<R>::C *__restrict__ clov,
                                                              const typename Vec<R>::T *__restrict__ in, typename Vec<R>::T *out)
{
    const unsigned j = blockIdx.x * DSLASH_BLOCK + threadIdx.x;
    if (j >= (unsigned)g.Vh * B) return;
    cx<R> x[12], y[12];
    load_spinor(in, j, x);
    clover_mul<R, false>(clov, j / B, x, y);
    store_spinor(out, j, y);
}

// explicit instantiation helper used by dslash_inst_*.cu
template <typename R, int B> int launch_dslash_B(const clover_ctx *ctx, const DslashArgs<R> &a, cudaStream_t st, int *grid_out);

}  // namespace clv
