// dslash2_kernel.cuh -- fp32 multi-rhs Wilson-clover stencil, one thread per (site, PAIR of right-hand sides).
//
// Same operator as dslash_kernel.cuh:  out = P ( X + coef * H_{p,1-p} in ).  Why a second mapping: at B = 8 the one-thread-per-
// (site, rhs) kernel is limited by the L1 data pipe (profiles/r1_dslash_ncu.md): every link / clover load is a broadcast -- the 8
// rhs-lanes of a site ask for the same 16 bytes, yet each quarter-warp costs a full wavefront -- so links carry 9 % of the bytes
// but 41 % of the wavefronts.  Here a thread owns two consecutive rhs of a site: the link and clover loads (and all the
// neighbour / address arithmetic) are issued once per pair, and the pair's spinor data, 32 contiguous bytes in the lane-blocked
// layout, moves with one 256-bit load or store (LDG.E.ENL2.256 on sm_100), so the spinor wavefronts per rhs do not grow.
#pragma once
#include "dslash_kernel.cuh"
#include <cuda_pipeline.h>

namespace clv {

#ifndef CLV_R2_MINB
#define CLV_R2_MINB 3
#endif
#ifndef CLV_R2_BLOCK_NODOT
#define CLV_R2_BLOCK_NODOT 32   // threads per CTA of the pair-kernel variants without dot products
#endif
#ifndef CLV_R2_BLOCK_DOT
#define CLV_R2_BLOCK_DOT 64   // threads per CTA of the pair-kernel variants that write a line of partial sums per CTA (128: +4 us per launch; 32: four times the lines for the scalar kernels, slower overall)
#endif
#ifndef CLV_R2_SMEM
#define CLV_R2_SMEM 1   // stage the CTA's clover blocks in shared memory with cp.async at kernel start
#endif

__device__ __forceinline__ void ldg256(const float4 *p, float4 &a, float4 &b)
{
    asm volatile("ld.global.nc.v8.f32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                 : "=f"(a.x), "=f"(a.y), "=f"(a.z), "=f"(a.w), "=f"(b.x), "=f"(b.y), "=f"(b.z), "=f"(b.w)
                 : "l"(p));
}
__device__ __forceinline__ void stg256(float4 *p, const float4 &a, const float4 &b)
{
    asm volatile("st.global.v8.f32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};" ::"l"(p), "f"(a.x), "f"(a.y), "f"(a.z), "f"(a.w), "f"(b.x), "f"(b.y),
                 "f"(b.z), "f"(b.w)
                 : "memory");
}

// spinors of rhs j and j+1 (j even): vectors (j, k) and (j+1, k) are adjacent 16-byte words
__device__ __forceinline__ void load_spinor2(const float4 *__restrict__ f, unsigned j, cx<float> a[12], cx<float> b[12])
{
    const float4 *p = f + lb_index(j, 0, 6);
#pragma unroll
    for (int k = 0; k < 6; k++) {
        float4 va, vb;
        ldg256(p + 32 * k, va, vb);
        a[2 * k] = mk<float>(va.x, va.y);
        a[2 * k + 1] = mk<float>(va.z, va.w);
        b[2 * k] = mk<float>(vb.x, vb.y);
        b[2 * k + 1] = mk<float>(vb.z, vb.w);
    }
}
__device__ __forceinline__ void store_spinor2(float4 *__restrict__ f, unsigned j, const cx<float> a[12], const cx<float> b[12])
{
    float4 *p = f + lb_index(j, 0, 6);
#pragma unroll
    for (int k = 0; k < 6; k++)
        stg256(p + 32 * k, make_float4(a[2 * k].re, a[2 * k].im, a[2 * k + 1].re, a[2 * k + 1].im),
               make_float4(b[2 * k].re, b[2 * k].im, b[2 * k + 1].re, b[2 * k + 1].im));
}

struct HopIn2 {
    cx<float> psiA[12], psiB[12];
    cx<float> u[9];
    bool neg;
};

template <int B, int RECON, int MU, int FWD>
__device__ __forceinline__ void hop_load2(const Geom &g, const OpData<float> &op, const float4 *__restrict__ in, int p, int cb, int rhs, const Coord &c,
                                          HopIn2 &d)
{
    bool wrap;
    const int nb = neighbour<MU, FWD>(g, cb, c, wrap);
    load_spinor2(in, (unsigned)nb * B + rhs, d.psiA, d.psiB);
    if (FWD) load_link<RECON>(p ? op.gauge[1][MU] : op.gauge[0][MU], cb, d.u);
    else load_link<RECON>(p ? op.gauge[0][MU] : op.gauge[1][MU], nb, d.u);
    d.neg = wrap && g.bc[MU] < 0;
}

template <int RECON, int MU, int FWD> __device__ __forceinline__ void hop_compute2(HopIn2 &d, HopAcc<float> &accA, HopAcc<float> &accB)
{
    cx<float> hA[6], hB[6];
    third_row<float, RECON>(d.u);
    project<float, MU, FWD>(d.psiA, hA);
    project<float, MU, FWD>(d.psiB, hB);
    if (d.neg) {
#pragma unroll
        for (int i = 0; i < 6; i++) {
            hA[i] = mk<float>(-hA[i].re, -hA[i].im);
            hB[i] = mk<float>(-hB[i].re, -hB[i].im);
        }
    }
    accA.template add<MU, FWD>(hA, d.u);
    accB.template add<MU, FWD>(hB, d.u);
}

// yA (+)= M xA, yB (+)= M xB with one load of the packed blocks; `srow` != nullptr: the site's 18 float4 rows staged in shared memory
template <bool ACCUM>
__device__ __forceinline__ void clover_mul2(const float2 *__restrict__ clov, unsigned cb, const float4 *srow, const cx<float> xA[12], cx<float> yA[12],
                                            const cx<float> xB[12], cx<float> yB[12])
{
#pragma unroll
    for (int blk = 0; blk < 2; blk++) {
        const int o = 6 * blk;
        cx<float> m[18];
        if (CLV_R2_SMEM) {
#pragma unroll
            for (int k = 0; k < 9; k++) {
                const float4 v = srow[9 * blk + k];
                m[2 * k] = mk<float>(v.x, v.y);
                m[2 * k + 1] = mk<float>(v.z, v.w);
            }
        } else load_clover_block(clov, cb, blk, m);
#pragma unroll
        for (int k = 0; k < 3; k++) {
            if (ACCUM) {
                yA[o + 2 * k] = yA[o + 2 * k] + m[k].re * xA[o + 2 * k];
                yA[o + 2 * k + 1] = yA[o + 2 * k + 1] + m[k].im * xA[o + 2 * k + 1];
                yB[o + 2 * k] = yB[o + 2 * k] + m[k].re * xB[o + 2 * k];
                yB[o + 2 * k + 1] = yB[o + 2 * k + 1] + m[k].im * xB[o + 2 * k + 1];
            } else {
                yA[o + 2 * k] = m[k].re * xA[o + 2 * k];
                yA[o + 2 * k + 1] = m[k].im * xA[o + 2 * k + 1];
                yB[o + 2 * k] = m[k].re * xB[o + 2 * k];
                yB[o + 2 * k + 1] = m[k].im * xB[o + 2 * k + 1];
            }
        }
        int k = 3;
#pragma unroll
        for (int i = 1; i < 6; i++)
#pragma unroll
            for (int j = 0; j < i; j++, k++) {
                fma_cx(yA[o + i], m[k], xA[o + j]);
                fma_conj(yA[o + j], m[k], xA[o + i]);
                fma_cx(yB[o + i], m[k], xB[o + j]);
                fma_conj(yB[o + j], m[k], xB[o + i]);
            }
    }
}

// per-rhs block reduction when a thread holds the partial sums of rhs 2q and 2q+1, q = threadIdx.x % (B/2); N = 3 sums per rhs
// into `partial`, or N = 7 (DOT_XW): sums 0..2 into `partial`, 3..6 into slots 0..3 of `partial2`
template <int B, int BLOCK, int N>
__device__ __forceinline__ void block_reduce_pair(double vA[N], double vB[N], double *__restrict__ partial, double *__restrict__ partial2)
{
    __shared__ double sm[BLOCK / 32][B][N];
#pragma unroll
    for (int off = 16; off >= B / 2 && off >= 1; off >>= 1) {
#pragma unroll
        for (int c = 0; c < N; c++) {
            vA[c] += __shfl_xor_sync(0xffffffffu, vA[c], off);
            vB[c] += __shfl_xor_sync(0xffffffffu, vB[c], off);
        }
    }
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (lane < B / 2) {
#pragma unroll
        for (int c = 0; c < N; c++) {
            sm[warp][2 * lane][c] = vA[c];
            sm[warp][2 * lane + 1][c] = vB[c];
        }
    }
    __syncthreads();
    if (threadIdx.x < B * N) {
        const int r = threadIdx.x / N, c = threadIdx.x % N;
        double s = 0;
#pragma unroll
        for (int w = 0; w < BLOCK / 32; w++) s += sm[w][r][c];
        if (c < 3) partial[((size_t)blockIdx.x * B + r) * 4 + c] = s;
        else partial2[((size_t)blockIdx.x * B + r) * 4 + (c - 3)] = s;
    }
}

// epilogue dot products of one rhs (same definitions as dslash_kernel).  The 12 terms of a site are summed in fp32 and converted
// once: the fp64 pipe and the F2F converter are slow enough that 12 conversions + 12 DADD per sum showed up in the kernel time
// (DOT_XW has seven sums); the accumulation across sites stays fp64.
template <int DOT> __device__ __forceinline__ void dots(const cx<float> acc[12], const cx<float> x[12], const cx<float> w[12], double *d)
{
    if (DOT == DOT_W) {
        float f0 = 0.f, f1 = 0.f;
#pragma unroll
        for (int i = 0; i < 12; i++) {  // <w, out>
            f0 += w[i].re * acc[i].re + w[i].im * acc[i].im;
            f1 += w[i].re * acc[i].im - w[i].im * acc[i].re;
        }
        d[0] += (double)f0;
        d[1] += (double)f1;
    }
    if (DOT == DOT_X || DOT == DOT_XW) {
        float f0 = 0.f, f1 = 0.f, f2 = 0.f;
#pragma unroll
        for (int i = 0; i < 12; i++) {  // <out, xin>, <out, out>
            f0 += acc[i].re * x[i].re + acc[i].im * x[i].im;
            f1 += acc[i].re * x[i].im - acc[i].im * x[i].re;
            f2 += acc[i].re * acc[i].re + acc[i].im * acc[i].im;
        }
        d[0] += (double)f0;
        d[1] += (double)f1;
        d[2] += (double)f2;
    }
    if (DOT == DOT_XW) {
        float f3 = 0.f, f4 = 0.f, f5 = 0.f, f6 = 0.f;
#pragma unroll
        for (int i = 0; i < 12; i++) {  // <w, out>, <w, xin>
            f3 += w[i].re * acc[i].re + w[i].im * acc[i].im;
            f4 += w[i].re * acc[i].im - w[i].im * acc[i].re;
            f5 += w[i].re * x[i].re + w[i].im * x[i].im;
            f6 += w[i].re * x[i].im - w[i].im * x[i].re;
        }
        d[3] += (double)f3;
        d[4] += (double)f4;
        d[5] += (double)f5;
        d[6] += (double)f6;
    }
}

// BLOCK threads per CTA, the register budget of 12 resident warps per SM whatever BLOCK is.  One-warp CTAs retire and refill
// the SM at a finer grain (A^-1 H: 225 -> 211 us at 24^3x48); variants with dot products keep 128 threads, because every CTA
// writes a line of partial sums that the scalar kernel must read back (four times as many CTAs cost more than they gain).
template <int B, int RECON, int XMODE, int PINV, int DOT, int BLOCK>
__global__ void __launch_bounds__(BLOCK, CLV_R2_MINB * DSLASH_BLOCK / BLOCK)
dslash2_kernel(const Geom g, const OpData<float> op, const DslashArgs<float> a)
{
    static_assert(B >= 2 && B % 2 == 0, "pairs of right-hand sides");
    const unsigned j = 2u * (blockIdx.x * BLOCK + threadIdx.x);   // first rhs of this thread's pair
    const bool active = j < (unsigned)g.Vh * B;
    constexpr int ND = DOT == DOT_XW ? 7 : 3;
    double dA[ND] = {}, dB[ND] = {};
    const int p = a.parity;
    constexpr int SITES = 2 * BLOCK / B;   // sites of this CTA: consecutive cb from blockIdx.x * SITES
    __shared__ __align__(16) float4 cl_s[(CLV_R2_SMEM && (XMODE == XM_CLOVER || PINV)) ? SITES * 18 : 1];
    if (CLV_R2_SMEM && (XMODE == XM_CLOVER || PINV)) {
        // the one clover field this variant needs (A for X = A x, A^-1 for P): 288 bytes per site, 16-byte async copies whose
        // DRAM latency is hidden behind the whole hop; consecutive threads copy consecutive sites of one row (coalesced)
        const float2 *clov = PINV ? (p ? op.clov_inv[1] : op.clov_inv[0]) : (p ? op.clov[1] : op.clov[0]);
        const float4 *base4 = reinterpret_cast<const float4 *>(clov);
        const unsigned cb0 = blockIdx.x * SITES;
        for (int item = threadIdx.x; item < SITES * 18; item += BLOCK) {
            const int row = item / SITES, site = item % SITES;
            const unsigned cbs = cb0 + site;
            if (cbs < (unsigned)g.Vh) __pipeline_memcpy_async(&cl_s[site * 18 + row], base4 + ((size_t)(cbs >> 5) * 18 + row) * 32 + (cbs & 31u), 16);
        }
        __pipeline_commit();
    }
    HopAcc<float> hA, hB;
    int cb = 0;
    if (active) {
        cb = j / B;
        const int rhs = j % B;
        const Coord c = decode(g, cb, p);
        hA.zero();
        hB.zero();
        prefetch_epilogue<float, (CLV_R2_SMEM && XMODE == XM_CLOVER ? XM_PLAIN : XMODE), (CLV_R2_SMEM ? 0 : PINV), DOT>(op, a, p, cb, j);   // x and w lines (the pair shares them)
        {
            HopIn2 d;
#define CLV_HOP2(MU, FW) hop_load2<B, RECON, MU, FW>(g, op, a.in, p, cb, rhs, c, d); hop_compute2<RECON, MU, FW>(d, hA, hB);
            CLV_HOP2(0, 1) CLV_HOP2(0, 0) CLV_HOP2(1, 1) CLV_HOP2(1, 0) CLV_HOP2(2, 1) CLV_HOP2(2, 0) CLV_HOP2(3, 1) CLV_HOP2(3, 0)
#undef CLV_HOP2
        }
    }
    if (CLV_R2_SMEM && (XMODE == XM_CLOVER || PINV)) {
        __pipeline_wait_prior(0);
        __syncthreads();
    }
    if (active) {
        const float4 *srow = cl_s + (cb - blockIdx.x * SITES) * 18;
        cx<float> accA[12], accB[12];
        hA.finish(accA);
        hB.finish(accB);
#pragma unroll
        for (int i = 0; i < 12; i++) {
            accA[i] = a.coef * accA[i];
            accB[i] = a.coef * accB[i];
        }
        cx<float> xA[12], xB[12];
        if (XMODE != XM_NONE) load_spinor2(a.xin, j, xA, xB);
        if (XMODE == XM_PLAIN) {
#pragma unroll
            for (int i = 0; i < 12; i++) {
                accA[i] = accA[i] + xA[i];
                accB[i] = accB[i] + xB[i];
            }
        }
        if (XMODE == XM_CLOVER) clover_mul2<true>(p ? op.clov[1] : op.clov[0], cb, srow, xA, accA, xB, accB);
        if (PINV) {
            cx<float> tA[12], tB[12];
            clover_mul2<false>(p ? op.clov_inv[1] : op.clov_inv[0], cb, srow, accA, tA, accB, tB);
#pragma unroll
            for (int i = 0; i < 12; i++) {
                accA[i] = tA[i];
                accB[i] = tB[i];
            }
        }
        cx<float> wA[12], wB[12];
        if (DOT == DOT_W || DOT == DOT_RES || DOT == DOT_S || DOT == DOT_XW) load_spinor2(a.w, j, wA, wB);
        if (DOT == DOT_RES) {  // result = w - acc, ||result||^2 (fp32 iteration precision: out32 and out are the same type here)
#pragma unroll
            for (int i = 0; i < 12; i++) {
                accA[i] = wA[i] - accA[i];
                accB[i] = wB[i] - accB[i];
                dA[0] += (double)accA[i].re * (double)accA[i].re + (double)accA[i].im * (double)accA[i].im;
                dB[0] += (double)accB[i].re * (double)accB[i].re + (double)accB[i].im * (double)accB[i].im;
            }
        }
        if (DOT != DOT_S) store_spinor2((DOT == DOT_RES && a.out32) ? a.out32 : a.out, j, accA, accB);
        if (DOT == DOT_S) {  // merged iteration: v stays in registers, out2 = s = w - alpha v with w = r
            const int rhs = j % B;
            const double2 alA = a.sc[rhs].alpha, alB = a.sc[rhs + 1].alpha;
            const cx<float> mA = mk<float>((float)-alA.x, (float)-alA.y), mB = mk<float>((float)-alB.x, (float)-alB.y);
#pragma unroll
            for (int i = 0; i < 12; i++) {
                fma_cx(wA[i], mA, accA[i]);
                fma_cx(wB[i], mB, accB[i]);
            }
            store_spinor2(a.out2, j, wA, wB);
        }
        dots<DOT>(accA, xA, wA, dA);
        dots<DOT>(accB, xB, wB, dB);
    }
    if (DOT != DOT_NONE && DOT != DOT_S) block_reduce_pair<B, BLOCK, ND>(dA, dB, a.partial, a.partial2);
}

}  // namespace clv
