// dslash3_kernel.cuh -- fp32 Wilson-clover stencil at B = 8: persistent one-warp (or two-warp) CTAs, operator data by bulk async copy.
//
// Same operator, thread mapping and arithmetic as dslash2_kernel.cuh (one thread per site and PAIR of right-hand sides, 256-bit
// spinor gathers straight into registers).  What changes is where the links and clover blocks come from.  In the pair kernel every
// direction waits for a link load that is a first-touch DRAM miss (links are 9 % of the bytes but none of them is ever re-used, so
// they never hit L2), with only 12 resident warps per SM to hide it (profiles/r1_tuning.md, "Ablations": removing the link loads
// took 23 % off the kernel).  Here the operator data of a CTA tile -- for each of its 8 sites the 8 links of the hop, stored site-major
// per OUTPUT site (context.h: pk_link), and the site's clover blocks -- is one contiguous record that a single thread fetches with
// cp.async.bulk (the TMA engine; SASS UBLKCP) into shared memory, completion on an mbarrier.  CTAs are persistent and the record of
// tile i+1 is in flight while tile i is computed, so the DRAM latency of the operator data is off the critical path of every
// direction and costs no registers; the links reach the registers by LDS right before their SU(3) product.
// The neighbour spinors are NOT staged: they would cross the shared-memory data path twice (profiles/r1_tuning.md, TMA-staged variant).
#pragma once
#include "dslash2_kernel.cuh"

namespace clv {

#ifndef CLV_R3_CTAS_PER_SM_WARPS
#define CLV_R3_CTAS_PER_SM_WARPS 12   // resident warps per SM (168 registers per thread)
#endif

__device__ __forceinline__ unsigned smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long *bar, unsigned count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long *bar, unsigned bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void *dst, const void *src, unsigned bytes, unsigned long long *bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst)), "l"(src), "r"(bytes),
                 "r"(smem_u32(bar))
                 : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long *bar, unsigned parity)
{
    asm volatile("{\n"
                 ".reg .pred P1;\n"
                 "LAB_WAIT:\n"
                 "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n"
                 "@P1 bra DONE;\n"
                 "bra LAB_WAIT;\n"
                 "DONE:\n"
                 "}\n" ::"r"(smem_u32(bar)),
                 "r"(parity)
                 : "memory");
}

// link d of a site record in shared memory (RECON floats each, consecutive): 16-byte loads where the offset allows
template <int RECON, int D> __device__ __forceinline__ void lds_link(const float *rec, cx<float> u[9])
{
    const float *q = rec + D * RECON;
    if (RECON == 12 || (D & 1) == 0) {   // 48 D or 144 (D/2) bytes: 16-byte aligned
#pragma unroll
        for (int k = 0; k < RECON / 4; k++) {
            const float4 v = *reinterpret_cast<const float4 *>(q + 4 * k);
            u[2 * k] = mk<float>(v.x, v.y);
            u[2 * k + 1] = mk<float>(v.z, v.w);
        }
        if (RECON == 18) {
            const float2 v = *reinterpret_cast<const float2 *>(q + 16);
            u[8] = mk<float>(v.x, v.y);
        }
    } else {   // 72 D bytes with D odd: 8 mod 16
        const float2 v0 = *reinterpret_cast<const float2 *>(q);
        u[0] = mk<float>(v0.x, v0.y);
#pragma unroll
        for (int k = 0; k < 4; k++) {
            const float4 v = *reinterpret_cast<const float4 *>(q + 2 + 4 * k);
            u[1 + 2 * k] = mk<float>(v.x, v.y);
            u[2 + 2 * k] = mk<float>(v.z, v.w);
        }
    }
}

template <int B, int MU, int FWD>
__device__ __forceinline__ void hop_gather3(const Geom &g, const float4 *__restrict__ in, int cb, int rhs, const Coord &c, HopIn2 &d)
{
    bool wrap;
    const int nb = neighbour<MU, FWD>(g, cb, c, wrap);
    load_spinor2(in, (unsigned)nb * B + rhs, d.psiA, d.psiB);
    d.neg = wrap && g.bc[MU] < 0;
}

template <int B, int RECON, int XMODE, int PINV, int DOT, int BLOCK>
__global__ void __launch_bounds__(BLOCK, CLV_R3_CTAS_PER_SM_WARPS * 32 / BLOCK)
dslash3_kernel(const Geom g, const OpData<float> op, const DslashArgs<float> a)
{
    static_assert(B >= 2 && B % 2 == 0, "pairs of right-hand sides");
    constexpr int SITES = 2 * BLOCK / B;          // sites of a CTA tile: consecutive cb
    constexpr int LREC = 8 * RECON;               // floats of a site's link record
    constexpr bool CLOV = (XMODE == XM_CLOVER || PINV);
    constexpr int ND = DOT == DOT_XW ? 7 : 3;
    __shared__ __align__(128) float lk_s[2][SITES * LREC];
    __shared__ __align__(128) float4 cl_s[2][CLOV ? SITES * 18 : 1];
    __shared__ __align__(8) unsigned long long bar[2];
    const int p = a.parity;
    const float *lk_g = p ? op.pk_link[1] : op.pk_link[0];
    const float *cl_g = PINV ? (p ? op.pk_clov_inv[1] : op.pk_clov_inv[0]) : (p ? op.pk_clov[1] : op.pk_clov[0]);
    const unsigned ntiles = ((unsigned)g.Vh + SITES - 1) / SITES;
    // one thread posts the record of a tile: links and (if this variant applies A or A^-1) clover blocks, one bulk copy each
    auto post = [&](unsigned tile, int buf) {
        const unsigned cb0 = tile * SITES, ns = min((unsigned)SITES, (unsigned)g.Vh - cb0);
        mbar_expect_tx(&bar[buf], ns * (LREC * 4u + (CLOV ? 288u : 0u)));
        bulk_g2s(&lk_s[buf][0], lk_g + (size_t)cb0 * LREC, ns * LREC * 4u, &bar[buf]);
        if (CLOV) bulk_g2s(&cl_s[buf][0], cl_g + (size_t)cb0 * 72, ns * 288u, &bar[buf]);
    };
    if (threadIdx.x == 0) {
        mbar_init(&bar[0], 1);
        mbar_init(&bar[1], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    if (threadIdx.x == 0 && blockIdx.x < ntiles) post(blockIdx.x, 0);
    double dA[ND] = {}, dB[ND] = {};
    unsigned it = 0;
    for (unsigned tile = blockIdx.x; tile < ntiles; tile += gridDim.x, it++) {
        const int buf = it & 1;
        if (threadIdx.x == 0 && tile + gridDim.x < ntiles) post(tile + gridDim.x, buf ^ 1);   // buf^1 was released by the barrier that ended iteration it-1
        const unsigned j = 2u * (tile * BLOCK + threadIdx.x);   // first rhs of this thread's pair
        const bool active = j < (unsigned)g.Vh * B;
        if (active) {
            const int cb = j / B, rhs = j % B;
            const int site = cb - tile * SITES;
            const Coord c = decode(g, cb, p);
            HopAcc<float> hA, hB;
            hA.zero();
            hB.zero();
            prefetch_epilogue<float, (XMODE == XM_CLOVER ? XM_PLAIN : XMODE), 0, DOT>(op, a, p, cb, j);   // x and w lines (the pair shares them)
            const float *rec = &lk_s[buf][site * LREC];
            {
                HopIn2 d;
                hop_gather3<B, 0, 1>(g, a.in, cb, rhs, c, d);
                mbar_wait(&bar[buf], (it >> 1) & 1);   // this tile's record has landed (posted one tile ahead)
#define CLV_HOP3(MU, FW) lds_link<RECON, 2 * MU + 1 - FW>(rec, d.u); hop_compute2<RECON, MU, FW>(d, hA, hB);
#define CLV_GAT3(MU, FW) hop_gather3<B, MU, FW>(g, a.in, cb, rhs, c, d);
                CLV_HOP3(0, 1) CLV_GAT3(0, 0) CLV_HOP3(0, 0) CLV_GAT3(1, 1) CLV_HOP3(1, 1) CLV_GAT3(1, 0) CLV_HOP3(1, 0)
                CLV_GAT3(2, 1) CLV_HOP3(2, 1) CLV_GAT3(2, 0) CLV_HOP3(2, 0) CLV_GAT3(3, 1) CLV_HOP3(3, 1) CLV_GAT3(3, 0) CLV_HOP3(3, 0)
#undef CLV_HOP3
#undef CLV_GAT3
            }
            const float4 *srow = &cl_s[buf][CLOV ? site * 18 : 0];
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
            if (XMODE == XM_CLOVER) clover_mul2<true>(nullptr, cb, srow, xA, accA, xB, accB);
            if (PINV) {
                cx<float> tA[12], tB[12];
                clover_mul2<false>(nullptr, cb, srow, accA, tA, accB, tB);
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
        } else {
            mbar_wait(&bar[buf], (it >> 1) & 1);
        }
        __syncthreads();   // every read of this tile's record is done before the buffer is posted again
    }
    // one line of partial sums per CTA for the whole launch (fixed tile -> CTA assignment and summation order: deterministic)
    if (DOT != DOT_NONE && DOT != DOT_S) block_reduce_pair<B, BLOCK, ND>(dA, dB, a.partial, a.partial2);
}

}  // namespace clv
