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
#ifndef CLV_DSLASH_MINB64
#define CLV_DSLASH_MINB64 2
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

// ---- accumulation of one direction: acc += (g, -+ B^+ g), g = U h or U^+ h --------------------------------------
// Generic (fp64) version: scalar complex arithmetic.
template <typename R> struct HopAcc {
    cx<R> acc[12];
    __device__ __forceinline__ void zero()
    {
#pragma unroll
        for (int i = 0; i < 12; i++) acc[i] = mk<R>(0, 0);
    }
    template <int MU, int FWD> __device__ __forceinline__ void add(const cx<R> h[6], const cx<R> u[9])
    {
        cx<R> gh[6];
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
    __device__ __forceinline__ void finish(cx<R> out[12]) const
    {
#pragma unroll
        for (int i = 0; i < 12; i++) out[i] = acc[i];
    }
};

// fp32 version on Blackwell's packed f32x2 pipe (FFMA2 / FADD2, one issue slot for two FMAs).  The two spin
// components of the half spinor are carried as a pair: the link acts on colour only, so each link element is a scalar
// broadcast operand of FFMA2 (SASS `R.F32`), and the SU(3) x half-spinor product costs 36 FFMA2 instead of 72 FFMA.
// Lower-spin accumulators are kept twice, in (2,3) order for mu = z,t and in (3,2) order for mu = x,y, so that
// B^+ g never needs a lane swap; they are merged in finish().
template <> struct HopAcc<float> {
    float2 ure[3], uim[3];  // (acc[a], acc[3+a])         real / imaginary parts
    float2 lre[3], lim[3];  // (acc[6+a], acc[9+a])       fed by mu = 2, 3
    float2 xre[3], xim[3];  // (acc[9+a], acc[6+a])       fed by mu = 0, 1
    __device__ __forceinline__ void zero()
    {
#pragma unroll
        for (int a = 0; a < 3; a++) ure[a] = uim[a] = lre[a] = lim[a] = xre[a] = xim[a] = make_float2(0.f, 0.f);
    }
    template <int MU, int FWD> __device__ __forceinline__ void add(const cx<float> h[6], const cx<float> u[9])
    {
        float2 hre[3], him[3];
#pragma unroll
        for (int b = 0; b < 3; b++) {
            hre[b] = make_float2(h[b].re, h[3 + b].re);
            him[b] = make_float2(h[b].im, h[3 + b].im);
        }
        constexpr float s = FWD ? -1.f : 1.f;
#pragma unroll
        for (int a = 0; a < 3; a++) {
            float2 gre, gim;
#pragma unroll
            for (int b = 0; b < 3; b++) {
                const cx<float> e = FWD ? u[a * 3 + b] : u[b * 3 + a];
                const float ei = FWD ? e.im : -e.im;  // U^+ : conjugate
                const float2 er2 = make_float2(e.re, e.re), ei2 = make_float2(ei, ei), nei2 = make_float2(-ei, -ei);
                if (b == 0) {
                    gre = __fmul2_rn(er2, hre[0]);
                    gim = __fmul2_rn(er2, him[0]);
                } else {
                    gre = __ffma2_rn(er2, hre[b], gre);
                    gim = __ffma2_rn(er2, him[b], gim);
                }
                gre = __ffma2_rn(nei2, him[b], gre);
                gim = __ffma2_rn(ei2, hre[b], gim);
            }
            ure[a] = __fadd2_rn(ure[a], gre);
            uim[a] = __fadd2_rn(uim[a], gim);
            if (MU == 0) {  // acc2 += s i g1, acc3 += s i g0
                xre[a] = __ffma2_rn(gim, make_float2(-s, -s), xre[a]);
                xim[a] = __ffma2_rn(gre, make_float2(s, s), xim[a]);
            } else if (MU == 1) {  // acc2 += s g1, acc3 -= s g0
                xre[a] = __ffma2_rn(gre, make_float2(-s, s), xre[a]);
                xim[a] = __ffma2_rn(gim, make_float2(-s, s), xim[a]);
            } else if (MU == 2) {  // acc2 += s i g0, acc3 -= s i g1
                lre[a] = __ffma2_rn(gim, make_float2(-s, s), lre[a]);
                lim[a] = __ffma2_rn(gre, make_float2(s, -s), lim[a]);
            } else {  // acc2 += s g0, acc3 += s g1
                lre[a] = __ffma2_rn(gre, make_float2(s, s), lre[a]);
                lim[a] = __ffma2_rn(gim, make_float2(s, s), lim[a]);
            }
        }
    }
    __device__ __forceinline__ void finish(cx<float> out[12]) const
    {
#pragma unroll
        for (int a = 0; a < 3; a++) {
            out[a] = mk<float>(ure[a].x, uim[a].x);
            out[3 + a] = mk<float>(ure[a].y, uim[a].y);
            out[6 + a] = mk<float>(lre[a].x + xre[a].y, lim[a].x + xim[a].y);
            out[9 + a] = mk<float>(lre[a].y + xre[a].x, lim[a].y + xim[a].x);
        }
    }
};

// One direction of the hop, split into its loads and its arithmetic so that the kernel can issue the loads of direction
// d+1 before the arithmetic of direction d (explicit software pipelining; profiles/r1_tuning.md).
template <typename R> struct HopIn {
    cx<R> psi[12];
    cx<R> u[9];
    bool neg;
};
template <typename R, int B, int RECON, int MU, int FWD>
__device__ __forceinline__ void hop_load(const Geom &g, const OpData<R> &op, const typename Vec<R>::T *__restrict__ in, int p, int cb, int rhs,
                                         const Coord &c, HopIn<R> &d)
{
    bool wrap;
    const int nb = neighbour<MU, FWD>(g, cb, c, wrap);
    load_spinor(in, (unsigned)nb * B + rhs, d.psi);
    // (ternaries rather than op.gauge[p]: runtime indexing of a kernel parameter would force a local copy)
    if (FWD) load_link<RECON>(p ? op.gauge[1][MU] : op.gauge[0][MU], cb, d.u);
    else load_link<RECON>(p ? op.gauge[0][MU] : op.gauge[1][MU], nb, d.u);
    d.neg = wrap && g.bc[MU] < 0;
}
template <typename R, int RECON, int MU, int FWD> __device__ __forceinline__ void hop_compute(HopIn<R> &d, HopAcc<R> &acc)
{
    cx<R> h[6];
    third_row<R, RECON>(d.u);
    project<R, MU, FWD>(d.psi, h);
    if (d.neg) {
#pragma unroll
        for (int i = 0; i < 6; i++) h[i] = mk<R>(-h[i].re, -h[i].im);
    }
    acc.template add<MU, FWD>(h, d.u);
}

// the 18 packed complex numbers of chirality block `blk` of one site (3 diagonal pairs, 15 lower off-diagonals)
__device__ __forceinline__ void load_clover_block(const double2 *__restrict__ clov, unsigned cb, int blk, cx<double> m[18])
{
    const double2 *p = clov + lb_index(cb, 18 * blk, 36);
#pragma unroll
    for (int k = 0; k < 18; k++) {
        double2 v = __ldg(p + 32 * k);
        m[k] = mk<double>(v.x, v.y);
    }
}
__device__ __forceinline__ void load_clover_block(const float2 *__restrict__ clov, unsigned cb, int blk, cx<float> m[18])
{
    const float4 *p = reinterpret_cast<const float4 *>(clov + (cb >> 5) * 32u * 36u) + (cb & 31u) + 32 * 9 * blk;
#pragma unroll
    for (int k = 0; k < 9; k++) {
        float4 v = __ldg(p + 32 * k);
        m[2 * k] = mk<float>(v.x, v.y);
        m[2 * k + 1] = mk<float>(v.z, v.w);
    }
}

// y (+)= M x for the two packed 6x6 Hermitian blocks of one site
template <typename R, bool ACCUM>
__device__ __forceinline__ void clover_mul(const typename Vec<R>::C *__restrict__ clov, unsigned cb, const cx<R> x[12], cx<R> y[12])
{
#pragma unroll
    for (int blk = 0; blk < 2; blk++) {
        const int o = 6 * blk;
        cx<R> m[18];
        load_clover_block(clov, cb, blk, m);
#pragma unroll
        for (int k = 0; k < 3; k++) {
            if (ACCUM) {
                y[o + 2 * k] = y[o + 2 * k] + m[k].re * x[o + 2 * k];
                y[o + 2 * k + 1] = y[o + 2 * k + 1] + m[k].im * x[o + 2 * k + 1];
            } else {
                y[o + 2 * k] = m[k].re * x[o + 2 * k];
                y[o + 2 * k + 1] = m[k].im * x[o + 2 * k + 1];
            }
        }
        int k = 3;
#pragma unroll
        for (int i = 1; i < 6; i++)
#pragma unroll
            for (int j = 0; j < i; j++, k++) {
                fma_cx(y[o + i], m[k], x[o + j]);
                fma_conj(y[o + j], m[k], x[o + i]);
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

// DOT_XW: seven sums per rhs; v[0..2] go to plane `partial` (slots 0..2), v[3..6] to plane `partial2` (slots 0..3)
template <int B, int BLOCK> __device__ __forceinline__ void block_reduce_rhs7(double v[7], double *__restrict__ partial, double *__restrict__ partial2)
{
    __shared__ double sm[BLOCK / 32][B][7];
#pragma unroll
    for (int off = 16; off >= B; off >>= 1) {
#pragma unroll
        for (int c = 0; c < 7; c++) v[c] += __shfl_xor_sync(0xffffffffu, v[c], off);
    }
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (lane < B) {
#pragma unroll
        for (int c = 0; c < 7; c++) sm[warp][lane][c] = v[c];
    }
    __syncthreads();
    if (threadIdx.x < B * 7) {
        const int r = threadIdx.x / 7, c = threadIdx.x % 7;
        double s = 0;
#pragma unroll
        for (int w = 0; w < BLOCK / 32; w++) s += sm[w][r][c];
        if (c < 3) partial[((size_t)blockIdx.x * B + r) * 4 + c] = s;
        else partial2[((size_t)blockIdx.x * B + r) * 4 + (c - 3)] = s;
    }
}

// L1 prefetch of everything the epilogue will read (clover blocks, xin, w): issued part-way through the hop so that the
// epilogue's loads -- first touches of DRAM lines, at the end of a dependent chain -- do not stall the warp for a full
// DRAM round trip with no registers left to overlap it.
#ifndef CLV_PIPE
#define CLV_PIPE 1
#endif
#ifndef CLV_PIPE64
#define CLV_PIPE64 0
#endif
__device__ __forceinline__ void prefetch_l1(const void *p) { asm volatile("prefetch.global.L1 [%0];" ::"l"(p)); }
template <typename R, int XMODE, int PINV, int DOT>
__device__ __forceinline__ void prefetch_epilogue(const OpData<R> &op, const DslashArgs<R> &a, int p, unsigned cb, unsigned j)
{
    constexpr int NV = Vec<R>::NV;
    if (XMODE != XM_NONE) {
        const typename Vec<R>::T *q = a.xin + lb_index(j, 0, NV);
#pragma unroll
        for (int k = 0; k < NV; k++) prefetch_l1(q + 32 * k);
    }
    if (DOT == DOT_W || DOT == DOT_RES || DOT == DOT_S || DOT == DOT_XW) {
        const typename Vec<R>::T *q = a.w + lb_index(j, 0, NV);
#pragma unroll
        for (int k = 0; k < NV; k++) prefetch_l1(q + 32 * k);
    }
    // clover rows are 16 bytes per lane in both precisions (float4 = two complex, double2 = one complex)
    constexpr int ROWS = (sizeof(R) == 4) ? 18 : 36;
    if (XMODE == XM_CLOVER) {
        const char *q = reinterpret_cast<const char *>(p ? op.clov[1] : op.clov[0]) + ((size_t)(cb >> 5) * ROWS * 32 + (cb & 31u)) * 16;
#pragma unroll
        for (int k = 0; k < ROWS; k++) prefetch_l1(q + 512 * k);
    }
    if (PINV) {
        const char *q = reinterpret_cast<const char *>(p ? op.clov_inv[1] : op.clov_inv[0]) + ((size_t)(cb >> 5) * ROWS * 32 + (cb & 31u)) * 16;
#pragma unroll
        for (int k = 0; k < ROWS; k++) prefetch_l1(q + 512 * k);
    }
}

// BLOCK threads per CTA at a fixed register budget per SM: one-warp CTAs for the variants without dot products (finer-grained
// refill of the SM: fp64 B = 8 -8 %, fp32 hop B = 8 -3 %), DSLASH_BLOCK where every CTA writes a line of partial sums.
#ifndef CLV_DSLASH_BLOCK_NODOT
#define CLV_DSLASH_BLOCK_NODOT 32
#endif
template <typename R, int B, int RECON, int XMODE, int PINV, int DOT, int BLOCK>
__global__ void __launch_bounds__(BLOCK, (sizeof(R) == 8 ? CLV_DSLASH_MINB64 : CLV_DSLASH_MINB) * DSLASH_BLOCK / BLOCK) dslash_kernel(const Geom g, const OpData<R> op, const DslashArgs<R> a)
{
    const unsigned j = blockIdx.x * BLOCK + threadIdx.x;
    const bool active = j < (unsigned)g.Vh * B;
    double d0 = 0, d1 = 0, d2 = 0, d3 = 0, d4 = 0, d5 = 0, d6 = 0;
    if (active) {
        const int cb = j / B, rhs = j % B, p = a.parity;
        const Coord c = decode(g, cb, p);
        HopAcc<R> hacc;
        hacc.zero();
        prefetch_epilogue<R, XMODE, PINV, DOT>(op, a, p, cb, j);
        // fp32: loads of direction d+1 are issued before the arithmetic of direction d (measured best with 128 registers);
        // fp64 has no registers to spare for that and runs the directions one after the other.
        if constexpr (sizeof(R) == 4 ? CLV_PIPE : CLV_PIPE64) {
        HopIn<R> hin0, hin1;
        hop_load<R, B, RECON, 0, 1>(g, op, a.in, p, cb, rhs, c, hin0);
        hop_load<R, B, RECON, 0, 0>(g, op, a.in, p, cb, rhs, c, hin1);
        hop_compute<R, RECON, 0, 1>(hin0, hacc);
        hop_load<R, B, RECON, 1, 1>(g, op, a.in, p, cb, rhs, c, hin0);
        hop_compute<R, RECON, 0, 0>(hin1, hacc);
        hop_load<R, B, RECON, 1, 0>(g, op, a.in, p, cb, rhs, c, hin1);
        hop_compute<R, RECON, 1, 1>(hin0, hacc);
        hop_load<R, B, RECON, 2, 1>(g, op, a.in, p, cb, rhs, c, hin0);
        hop_compute<R, RECON, 1, 0>(hin1, hacc);
        hop_load<R, B, RECON, 2, 0>(g, op, a.in, p, cb, rhs, c, hin1);
        hop_compute<R, RECON, 2, 1>(hin0, hacc);
        hop_load<R, B, RECON, 3, 1>(g, op, a.in, p, cb, rhs, c, hin0);
        hop_compute<R, RECON, 2, 0>(hin1, hacc);
        hop_load<R, B, RECON, 3, 0>(g, op, a.in, p, cb, rhs, c, hin1);
        hop_compute<R, RECON, 3, 1>(hin0, hacc);
        hop_compute<R, RECON, 3, 0>(hin1, hacc);
        } else
        {
            HopIn<R> d;
#define CLV_HOP(MU, FW) hop_load<R, B, RECON, MU, FW>(g, op, a.in, p, cb, rhs, c, d); hop_compute<R, RECON, MU, FW>(d, hacc);
            CLV_HOP(0, 1) CLV_HOP(0, 0) CLV_HOP(1, 1) CLV_HOP(1, 0) CLV_HOP(2, 1) CLV_HOP(2, 0) CLV_HOP(3, 1) CLV_HOP(3, 0)
#undef CLV_HOP
        }
        cx<R> acc[12];
        hacc.finish(acc);
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
        if (DOT == DOT_RES) {  // residual epilogue: result = w - acc, ||result||^2, stored in the iteration precision
            cx<R> w[12];
            load_spinor(a.w, j, w);
#pragma unroll
            for (int i = 0; i < 12; i++) {
                acc[i] = w[i] - acc[i];
                d0 += (double)acc[i].re * (double)acc[i].re + (double)acc[i].im * (double)acc[i].im;
            }
            if (a.out32) {
                cx<float> f[12];
#pragma unroll
                for (int i = 0; i < 12; i++) f[i] = mk<float>((float)acc[i].re, (float)acc[i].im);
                store_spinor(a.out32, j, f);
            } else if (a.out) store_spinor(a.out, j, acc);   // neither: only the norm is wanted (final verification)
        } else if (DOT != DOT_S) store_spinor(a.out, j, acc);
        if (DOT == DOT_S) {  // merged iteration: v stays in registers, out2 = s = w - alpha v with w = r
            cx<R> w[12];
            load_spinor(a.w, j, w);
            const double2 al = a.sc[rhs].alpha;
            const cx<R> mal = mk<R>((R)-al.x, (R)-al.y);
#pragma unroll
            for (int i = 0; i < 12; i++) fma_cx(w[i], mal, acc[i]);
            store_spinor(a.out2, j, w);
        }
        // dot products: the 12 terms of a site are summed in the kernel's precision and converted once (fp32: the F2F converter
        // and the fp64 pipe are slow); the accumulation across sites is fp64
        if (DOT == DOT_XW) {  // merged iteration: <out,xin>, <out,out>, <w,out>, <w,xin> with out = t, xin = s, w = r0
            cx<R> w[12];
            load_spinor(a.w, j, w);
            R f0 = 0, f1 = 0, f2 = 0, f3 = 0, f4 = 0, f5 = 0, f6 = 0;
#pragma unroll
            for (int i = 0; i < 12; i++) {
                f0 += acc[i].re * x[i].re + acc[i].im * x[i].im;
                f1 += acc[i].re * x[i].im - acc[i].im * x[i].re;
                f2 += acc[i].re * acc[i].re + acc[i].im * acc[i].im;
                f3 += w[i].re * acc[i].re + w[i].im * acc[i].im;
                f4 += w[i].re * acc[i].im - w[i].im * acc[i].re;
                f5 += w[i].re * x[i].re + w[i].im * x[i].im;
                f6 += w[i].re * x[i].im - w[i].im * x[i].re;
            }
            d0 = (double)f0; d1 = (double)f1; d2 = (double)f2; d3 = (double)f3; d4 = (double)f4; d5 = (double)f5; d6 = (double)f6;
        }
        if (DOT == DOT_W) {
            cx<R> w[12];
            load_spinor(a.w, j, w);
            R f0 = 0, f1 = 0;
#pragma unroll
            for (int i = 0; i < 12; i++) {  // <w, out> = sum conj(w) out
                f0 += w[i].re * acc[i].re + w[i].im * acc[i].im;
                f1 += w[i].re * acc[i].im - w[i].im * acc[i].re;
            }
            d0 = (double)f0; d1 = (double)f1;
        }
        if (DOT == DOT_X) {
            R f0 = 0, f1 = 0, f2 = 0;
#pragma unroll
            for (int i = 0; i < 12; i++) {  // <out, xin> and <out, out>
                f0 += acc[i].re * x[i].re + acc[i].im * x[i].im;
                f1 += acc[i].re * x[i].im - acc[i].im * x[i].re;
                f2 += acc[i].re * acc[i].re + acc[i].im * acc[i].im;
            }
            d0 = (double)f0; d1 = (double)f1; d2 = (double)f2;
        }
    }
    if (DOT == DOT_XW) {
        double d[7] = {d0, d1, d2, d3, d4, d5, d6};
        block_reduce_rhs7<B, BLOCK>(d, a.partial, a.partial2);
    } else if (DOT != DOT_NONE && DOT != DOT_S) block_reduce_rhs<B, BLOCK>(d0, d1, d2, a.partial);
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
