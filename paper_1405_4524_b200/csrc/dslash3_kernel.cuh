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

#ifndef CLV_R3_PFT
#define CLV_R3_PFT 1   // L2 prefetch of the tile's forward-t neighbour lines when the tile starts
#endif
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

// (Own-site streams of the epilogue, x and w: no prefetch.  The pair kernel prefetches them into L1 at kernel start; here the L1 is smaller by the
// record buffers and the lines do not survive the hop: measured at 24^3x48, s epilogue 254 us with, 245 us without; into L2: 255 us.)
__device__ __forceinline__ void prefetch_l2(const void *p) { asm volatile("prefetch.global.L2 [%0];" ::"l"(p)); }

// yA (+)= M xA, yB (+)= M xB for the two packed 6x6 Hermitian blocks of a site (rows `srow` in shared memory), on the packed f32x2 pipe: the two
// right-hand sides of the thread ride in the two halves of an FFMA2 and the matrix element is its broadcast operand, so the 504 flop of a
// clover product cost 126 FFMA2 + 12 FMUL2 per rhs pair instead of 480 FFMA + 24 FMUL (a three-register FFMA and an FFMA2 hold the FP32 pipe equally long).
#ifndef CLV_R3_CLOVER_PACKED
#define CLV_R3_CLOVER_PACKED 1
#endif
template <bool ACCUM>
__device__ __forceinline__ void clover_mul2_packed(const float4 *srow, const cx<float> xA[12], cx<float> yA[12], const cx<float> xB[12], cx<float> yB[12])
{
#pragma unroll
    for (int blk = 0; blk < 2; blk++) {
        const int o = 6 * blk;
        cx<float> m[18];
#pragma unroll
        for (int k = 0; k < 9; k++) {
            const float4 v = srow[9 * blk + k];
            m[2 * k] = mk<float>(v.x, v.y);
            m[2 * k + 1] = mk<float>(v.z, v.w);
        }
        float2 xr[6], xi[6], yr[6], yi[6];
#pragma unroll
        for (int i = 0; i < 6; i++) {
            xr[i] = make_float2(xA[o + i].re, xB[o + i].re);
            xi[i] = make_float2(xA[o + i].im, xB[o + i].im);
            if (ACCUM) {
                yr[i] = make_float2(yA[o + i].re, yB[o + i].re);
                yi[i] = make_float2(yA[o + i].im, yB[o + i].im);
            }
        }
#pragma unroll
        for (int k = 0; k < 3; k++) {   // real diagonal entries (2k, 2k) = m[k].re and (2k+1, 2k+1) = m[k].im
            const float2 d0 = make_float2(m[k].re, m[k].re), d1 = make_float2(m[k].im, m[k].im);
            if (ACCUM) {
                yr[2 * k] = __ffma2_rn(d0, xr[2 * k], yr[2 * k]);
                yi[2 * k] = __ffma2_rn(d0, xi[2 * k], yi[2 * k]);
                yr[2 * k + 1] = __ffma2_rn(d1, xr[2 * k + 1], yr[2 * k + 1]);
                yi[2 * k + 1] = __ffma2_rn(d1, xi[2 * k + 1], yi[2 * k + 1]);
            } else {
                yr[2 * k] = __fmul2_rn(d0, xr[2 * k]);
                yi[2 * k] = __fmul2_rn(d0, xi[2 * k]);
                yr[2 * k + 1] = __fmul2_rn(d1, xr[2 * k + 1]);
                yi[2 * k + 1] = __fmul2_rn(d1, xi[2 * k + 1]);
            }
        }
        int k = 3;
#pragma unroll
        for (int i = 1; i < 6; i++)
#pragma unroll
            for (int j = 0; j < i; j++, k++) {
                const float2 mr = make_float2(m[k].re, m[k].re), mi = make_float2(m[k].im, m[k].im), nmi = make_float2(-m[k].im, -m[k].im);
                // y[i] += m x[j]
                yr[i] = __ffma2_rn(mr, xr[j], yr[i]);
                yr[i] = __ffma2_rn(nmi, xi[j], yr[i]);
                yi[i] = __ffma2_rn(mr, xi[j], yi[i]);
                yi[i] = __ffma2_rn(mi, xr[j], yi[i]);
                // y[j] += conj(m) x[i]
                yr[j] = __ffma2_rn(mr, xr[i], yr[j]);
                yr[j] = __ffma2_rn(mi, xi[i], yr[j]);
                yi[j] = __ffma2_rn(mr, xi[i], yi[j]);
                yi[j] = __ffma2_rn(nmi, xr[i], yi[j]);
            }
#pragma unroll
        for (int i = 0; i < 6; i++) {
            yA[o + i] = mk<float>(yr[i].x, yi[i].x);
            yB[o + i] = mk<float>(yr[i].y, yi[i].y);
        }
    }
}

// per-tile partial sums of one rhs in fp32 (the 12 terms of a site; same definitions as dots<> in dslash2_kernel.cuh)
template <int DOT> __device__ __forceinline__ void dots_f(const cx<float> acc[12], const cx<float> x[12], const cx<float> w[12], float *f)
{
    if (DOT == DOT_W) {
        float f0 = 0.f, f1 = 0.f;
#pragma unroll
        for (int i = 0; i < 12; i++) {  // <w, out>
            f0 += w[i].re * acc[i].re + w[i].im * acc[i].im;
            f1 += w[i].re * acc[i].im - w[i].im * acc[i].re;
        }
        f[0] = f0; f[1] = f1; f[2] = 0.f;
    }
    if (DOT == DOT_RES) {  // acc already holds w - (...)
        float f0 = 0.f;
#pragma unroll
        for (int i = 0; i < 12; i++) f0 += acc[i].re * acc[i].re + acc[i].im * acc[i].im;
        f[0] = f0; f[1] = 0.f; f[2] = 0.f;
    }
    if (DOT == DOT_X || DOT == DOT_XW) {
        float f0 = 0.f, f1 = 0.f, f2 = 0.f;
#pragma unroll
        for (int i = 0; i < 12; i++) {  // <out, xin>, <out, out>
            f0 += acc[i].re * x[i].re + acc[i].im * x[i].im;
            f1 += acc[i].re * x[i].im - acc[i].im * x[i].re;
            f2 += acc[i].re * acc[i].re + acc[i].im * acc[i].im;
        }
        f[0] = f0; f[1] = f1; f[2] = f2;
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
        f[3] = f3; f[4] = f4; f[5] = f5; f[6] = f6;
    }
}

// Reduce-scatter of a warp tile's partial sums (B = 8, one-warp CTAs: lane = 4 site + pair, 8 sites x 4 rhs pairs).  v holds the NV = 2 ND
// sums of this thread's two rhs, padded to 8 K values (K = 1 | 2).  Three butterfly steps over the site bits of the lane, each sending one
// half of the values and keeping the other, leave lane (site s, pair q) with the sums over the tile's 8 sites of values K s .. K s + K - 1 of
// pair q: 7 or 14 shuffles instead of 3 NV, and K values per thread to store instead of NV.
// (The 8 sites of a tile are summed in fp32; the tiles' lines are added in fp64 by the scalar kernel in a fixed order: deterministic.)
template <int K> __device__ __forceinline__ void reduce_scatter_sites(float (&v)[8 * K], float (&out)[K])
{
    const unsigned lane = threadIdx.x & 31u;
    float h4[4 * K], h2[2 * K];
    {
        const bool up = lane & 16u;
#pragma unroll
        for (int i = 0; i < 4 * K; i++) {
            const float send = up ? v[i] : v[4 * K + i], keep = up ? v[4 * K + i] : v[i];
            h4[i] = keep + __shfl_xor_sync(0xffffffffu, send, 16);
        }
    }
    {
        const bool up = lane & 8u;
#pragma unroll
        for (int i = 0; i < 2 * K; i++) {
            const float send = up ? h4[i] : h4[2 * K + i], keep = up ? h4[2 * K + i] : h4[i];
            h2[i] = keep + __shfl_xor_sync(0xffffffffu, send, 8);
        }
    }
    {
        const bool up = lane & 4u;
#pragma unroll
        for (int i = 0; i < K; i++) {
            const float send = up ? h2[i] : h2[K + i], keep = up ? h2[K + i] : h2[i];
            out[i] = keep + __shfl_xor_sync(0xffffffffu, send, 4);
        }
    }
}

// The CTA (one warp: 8 consecutive sites x 4 rhs pairs) loops over tiles.  The link records are double-buffered (the next tile's are posted when
// a tile starts); the clover records have ONE buffer, re-posted for the next tile as soon as this tile's A / A^-1 product has read it -- the
// copy then has the whole hop of the next tile to land.  Shared memory is kept small on purpose: what the records do not take stays L1, and
// L1 capacity bounds the bytes the gathers can have in flight (measured at 24^3x48: the same kernel with 32 instead of 64 KB of L1 is 25 %
// slower).  Tiles are handed out in order by an atomic counter (`sched[0]`; the first gridDim.x tiles statically), not round-robin: CTAs
// that fall behind would otherwise spread the window of sites in flight over many timeslices and the neighbour gathers would stop hitting L2
// (measured at 32^3x64: a round-robin assignment lost everything the records had gained).  The last CTA to leave re-arms the counters for
// the next launch.  Dot-product variants write one line of partial sums per tile (the sums of the tile's 8 sites).
#ifndef CLV_R3_CBUF
#define CLV_R3_CBUF 1
#endif
#ifndef CLV_R3_LBUF
#define CLV_R3_LBUF 2
#endif
template <int B, int RECON, int XMODE, int PINV, int DOT, int BLOCK>
__global__ void __launch_bounds__(BLOCK, CLV_R3_CTAS_PER_SM_WARPS * 32 / BLOCK)
dslash3_kernel(const Geom g, const OpData<float> op, const DslashArgs<float> a, unsigned *__restrict__ sched)
{
    static_assert(B == 8 && BLOCK == 32, "lane = 4 site + pair");
    constexpr int SITES = 2 * BLOCK / B;          // sites of a CTA tile: consecutive cb
    constexpr int LREC = pk_link_stride(RECON);   // floats of a site's (padded) link record
    constexpr int CREC = PK_CLOV_STRIDE;          // floats of a site's (padded) clover record
    constexpr bool CLOV = (XMODE == XM_CLOVER || PINV);
    constexpr bool RED = (DOT != DOT_NONE && DOT != DOT_S);
    constexpr int ND = DOT == DOT_XW ? 7 : 3;     // sums per rhs
    constexpr int K = DOT == DOT_XW ? 2 : 1;      // accumulators per thread after the reduce-scatter: values K s .. K s + K - 1 of (2 ND padded to 8 K)
    constexpr int NCB = CLV_R3_CBUF;              // clover buffers
    constexpr int NLB = CLV_R3_LBUF;              // link buffers
    __shared__ __align__(128) float lk_s[NLB][SITES * LREC];
    __shared__ __align__(128) float cl_s[NCB][CLOV ? SITES * CREC : 4];
    __shared__ __align__(8) unsigned long long bar[2], bar_c[NCB];
    __shared__ unsigned next_s[2];
    const int p = a.parity;
    const float *lk_g = p ? op.pk_link[1] : op.pk_link[0];
    const float *cl_g = PINV ? (p ? op.pk_clov_inv[1] : op.pk_clov_inv[0]) : (p ? op.pk_clov[1] : op.pk_clov[0]);
    const unsigned ntiles = ((unsigned)g.Vh + SITES - 1) / SITES;
    // one thread posts the records of a tile with one bulk copy each
    auto post_links = [&](unsigned tile, int buf) {
        const unsigned cb0 = tile * SITES, ns = min((unsigned)SITES, (unsigned)g.Vh - cb0);
        mbar_expect_tx(&bar[buf], ns * LREC * 4u);
        bulk_g2s(&lk_s[buf][0], lk_g + (size_t)cb0 * LREC, ns * LREC * 4u, &bar[buf]);
    };
    auto post_clover = [&](unsigned tile, int buf) {
        const unsigned cb0 = tile * SITES, ns = min((unsigned)SITES, (unsigned)g.Vh - cb0);
        mbar_expect_tx(&bar_c[buf], ns * CREC * 4u);
        bulk_g2s(&cl_s[buf][0], cl_g + (size_t)cb0 * CREC, ns * CREC * 4u, &bar_c[buf]);
    };
    if (threadIdx.x == 0) {
        mbar_init(&bar[0], 1);
        mbar_init(&bar[1], 1);
#pragma unroll
        for (int k = 0; k < NCB; k++) mbar_init(&bar_c[k], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    unsigned it = 0, tile = blockIdx.x;   // (the grid never exceeds the tiles)
    if (threadIdx.x == 0) {
        post_links(tile, 0);
        if (CLOV) post_clover(tile, 0);
    }
    do {
        const int buf = it & 1, cbuf = NCB == 2 ? buf : 0, lbuf = NLB == 2 ? buf : 0;
        const unsigned par = (it >> 1) & 1, cpar = NCB == 2 ? par : (it & 1), lpar = NLB == 2 ? par : (it & 1);
        if (threadIdx.x == 0) {   // draw the next tile and post its links; buf^1 was released by the barrier that ended iteration it-1
            // (drawing the ticket one tile earlier, so that nobody waits for the atomic, measured 2 % slower)
            const unsigned nt = gridDim.x + atomicAdd(&sched[0], 1u);
            next_s[buf] = nt;
            if (nt < ntiles) {
                if (NLB == 2) post_links(nt, buf ^ 1);
                if (CLOV && NCB == 2) post_clover(nt, buf ^ 1);
            }
        }
        const unsigned j = 2u * (tile * BLOCK + threadIdx.x);   // first rhs of this thread's pair
        const bool active = j < (unsigned)g.Vh * B;
        const int cb = j / B, rhs = j % B;
        const int site = cb - tile * SITES;
        float v[8 * K] = {};
        cx<float> accA[12], accB[12], xA[12], xB[12];
        if (active) {
            const Coord c = decode(g, cb, p);
            HopAcc<float> hA, hB;
            hA.zero();
            hB.zero();
            if (CLV_R3_PFT) {
                // Tiles are processed in order of cb (t slowest), so the forward-t neighbours are the frontier: nobody has read them yet
                // and their gather, the seventh direction, is a DRAM miss.  Ask L2 for their lines now: lane (site, pair q) takes rows
                // q, q + 4 of its site's neighbour.  (Measured: -4 %; the same for the next tile, or for the own-site streams: slower.)
                bool wrap;
                const int nbt = neighbour<3, 1>(g, cb, c, wrap);
                const float4 *q4 = a.in + lb_index((unsigned)nbt * B, 0, 6);
                const int q = rhs >> 1;
                prefetch_l2(q4 + 32 * q);
                if (q < 2) prefetch_l2(q4 + 32 * (q + 4));
            }
            const float *rec = &lk_s[lbuf][site * LREC];
            {
                HopIn2 d;
                hop_gather3<B, 0, 1>(g, a.in, cb, rhs, c, d);
                mbar_wait(&bar[lbuf], lpar);   // this tile's links have landed (posted one tile ahead)
#define CLV_HOP3(MU, FW) lds_link<RECON, 2 * MU + 1 - FW>(rec, d.u); hop_compute2<RECON, MU, FW>(d, hA, hB);
#define CLV_GAT3(MU, FW) hop_gather3<B, MU, FW>(g, a.in, cb, rhs, c, d);
                CLV_HOP3(0, 1) CLV_GAT3(0, 0) CLV_HOP3(0, 0) CLV_GAT3(1, 1) CLV_HOP3(1, 1) CLV_GAT3(1, 0) CLV_HOP3(1, 0)
                CLV_GAT3(2, 1) CLV_HOP3(2, 1) CLV_GAT3(2, 0) CLV_HOP3(2, 0) CLV_GAT3(3, 1) CLV_HOP3(3, 1) CLV_GAT3(3, 0) CLV_HOP3(3, 0)
#undef CLV_HOP3
#undef CLV_GAT3
            }
            hA.finish(accA);
            hB.finish(accB);
#pragma unroll
            for (int i = 0; i < 12; i++) {
                accA[i] = a.coef * accA[i];
                accB[i] = a.coef * accB[i];
            }
            if (XMODE != XM_NONE) load_spinor2(a.xin, j, xA, xB);
            if (XMODE == XM_PLAIN) {
#pragma unroll
                for (int i = 0; i < 12; i++) {
                    accA[i] = accA[i] + xA[i];
                    accB[i] = accB[i] + xB[i];
                }
            }
            if (CLOV) {
                mbar_wait(&bar_c[cbuf], cpar);
                const float4 *srow = reinterpret_cast<const float4 *>(&cl_s[cbuf][site * CREC]);
                // (packed form for the A^-1 product only: measured at 24^3x48, A^-1 H 176 -> 170 us; for y += A x it costs more moves than it saves: +3-5 %)
                if (XMODE == XM_CLOVER) clover_mul2<true>(nullptr, cb, srow, xA, accA, xB, accB);
                if (PINV) {
                    cx<float> tA[12], tB[12];
                    if (CLV_R3_CLOVER_PACKED) clover_mul2_packed<false>(srow, accA, tA, accB, tB);
                    else clover_mul2<false>(nullptr, cb, srow, accA, tA, accB, tB);
#pragma unroll
                    for (int i = 0; i < 12; i++) {
                        accA[i] = tA[i];
                        accB[i] = tB[i];
                    }
                }
            }
        } else {
            mbar_wait(&bar[lbuf], lpar);
            if (CLOV) mbar_wait(&bar_c[cbuf], cpar);
        }
        if ((CLOV && NCB == 1) || NLB == 1) {   // the clover buffer has been read: it takes the next tile's blocks while this tile is finished and the next one hops
            __syncthreads();
            if (threadIdx.x == 0 && next_s[buf] < ntiles) {
                if (NLB == 1) post_links(next_s[buf], 0);
                if (CLOV && NCB == 1) post_clover(next_s[buf], 0);
            }
        }
        if (active) {
            cx<float> wA[12], wB[12];
            if (DOT == DOT_W || DOT == DOT_RES || DOT == DOT_S || DOT == DOT_XW) load_spinor2(a.w, j, wA, wB);
            if (DOT == DOT_RES) {  // result = w - acc (fp32 iteration precision: out32 and out are the same type here)
#pragma unroll
                for (int i = 0; i < 12; i++) {
                    accA[i] = wA[i] - accA[i];
                    accB[i] = wB[i] - accB[i];
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
            if (RED) {
                dots_f<DOT>(accA, xA, wA, v);
                dots_f<DOT>(accB, xB, wB, v + ND);
            }
        }
        if (RED) {   // one line of partial sums per TILE, indexed by the tile: the scalar kernel adds the lines in a fixed order, so the
            // result does not depend on which CTA the scheduler gave the tile to (solves stay bit-reproducible)
            float t[K];
            reduce_scatter_sites<K>(v, t);
            // lane (site s, pair q) holds values K s .. K s + K - 1 of pair q: value c < ND belongs to rhs 2q, else c - ND to rhs 2q + 1
            const int s = threadIdx.x >> 2, q = threadIdx.x & 3;
#pragma unroll
            for (int k = 0; k < K; k++) {
                const int cidx = K * s + k;
                if (cidx < 2 * ND) {
                    const int r = 2 * q + (cidx >= ND), cc = cidx % ND;
                    if (cc < 3) a.partial[((size_t)tile * B + r) * 4 + cc] = (double)t[k];
                    else a.partial2[((size_t)tile * B + r) * 4 + (cc - 3)] = (double)t[k];
                }
            }
        }
        __syncthreads();   // every read of this tile's link records is done before the buffer is posted again
        tile = next_s[buf];
        it++;
    } while (tile < ntiles);
    if (threadIdx.x == 0) {   // the last CTA to finish re-arms the tile counter for the next launch on this context
        __threadfence();
        if (atomicInc(&sched[1], gridDim.x - 1) == gridDim.x - 1) sched[0] = 0;
    }
}

}  // namespace clv
