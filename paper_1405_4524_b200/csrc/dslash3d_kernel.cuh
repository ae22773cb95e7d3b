// dslash3d_kernel.cuh -- fp64 Wilson-clover stencil at B = 8 for the fp64 steps of the mixed-precision solve (source preparation, reliable
// updates, odd-site reconstruction, full-lattice verification): the design of dslash3_kernel.cuh with one thread per (site, rhs).
//
// A one-warp CTA owns tiles of 4 consecutive sites x 8 right-hand sides (lane = 8 site + rhs: a warp's 16-byte spinor loads are 4 full
// 128-byte lines).  The operator data of a tile -- the 8 links per site of the hop, site-major per OUTPUT site, and the site's clover
// blocks, both in fp64 -- is fetched by one thread with cp.async.bulk into shared memory, links double-buffered one tile ahead, clover
// single-buffered and re-posted once read; CTAs are persistent, tiles handed out in order by an atomic counter; the forward-t frontier
// is prefetched into L2.  Only the variants the mixed solve launches are built here (dslash_inst.cuh falls back to dslash_kernel for the rest).
#pragma once
#include "dslash3_kernel.cuh"

namespace clv {

#ifndef CLV_R3D_WARPS_PER_SM
#define CLV_R3D_WARPS_PER_SM 8   // 255 registers per thread
#endif

// link d of a site record in shared memory (9 double2, consecutive)
template <int D> __device__ __forceinline__ void lds_link64(const double *rec, cx<double> u[9])
{
    const double2 *q = reinterpret_cast<const double2 *>(rec + D * 18);
#pragma unroll
    for (int k = 0; k < 9; k++) {
        const double2 v = q[k];
        u[k] = mk<double>(v.x, v.y);
    }
}

// y (+)= M x for the two packed 6x6 Hermitian blocks of one site, the 36 double2 rows read from shared memory
template <bool ACCUM> __device__ __forceinline__ void clover_mul_rows(const double2 *srow, const cx<double> x[12], cx<double> y[12])
{
#pragma unroll
    for (int blk = 0; blk < 2; blk++) {
        const int o = 6 * blk;
        cx<double> m[18];
#pragma unroll
        for (int k = 0; k < 18; k++) {
            const double2 v = srow[18 * blk + k];
            m[k] = mk<double>(v.x, v.y);
        }
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

template <int XMODE, int PINV, int DOT>
__global__ void __launch_bounds__(32, CLV_R3D_WARPS_PER_SM)
dslash3d_kernel(const Geom g, const OpData<double> op, const DslashArgs<double> a, unsigned *__restrict__ sched)
{
    static_assert(DOT == DOT_NONE || DOT == DOT_RES, "variants of the mixed-precision solve only");
    constexpr int B = 8, SITES = 4;
    constexpr int LREC = pk_link_stride(18);      // doubles of a site's (padded) link record
    constexpr int CREC = PK_CLOV_STRIDE;          // doubles of a site's (padded) clover record
    constexpr bool CLOV = (XMODE == XM_CLOVER || PINV);
    __shared__ __align__(128) double lk_s[2][SITES * LREC];
    __shared__ __align__(128) double cl_s[CLOV ? SITES * CREC : 2];
    __shared__ __align__(8) unsigned long long bar[2], bar_c;
    __shared__ unsigned next_s[2];
    const int p = a.parity;
    const double *lk_g = p ? op.pk_link[1] : op.pk_link[0];
    const double *cl_g = PINV ? (p ? op.pk_clov_inv[1] : op.pk_clov_inv[0]) : (p ? op.pk_clov[1] : op.pk_clov[0]);
    const unsigned ntiles = ((unsigned)g.Vh + SITES - 1) / SITES;
    auto post_links = [&](unsigned tile, int buf) {
        const unsigned cb0 = tile * SITES, ns = min((unsigned)SITES, (unsigned)g.Vh - cb0);
        mbar_expect_tx(&bar[buf], ns * LREC * 8u);
        bulk_g2s(&lk_s[buf][0], lk_g + (size_t)cb0 * LREC, ns * LREC * 8u, &bar[buf]);
    };
    auto post_clover = [&](unsigned tile) {
        const unsigned cb0 = tile * SITES, ns = min((unsigned)SITES, (unsigned)g.Vh - cb0);
        mbar_expect_tx(&bar_c, ns * CREC * 8u);
        bulk_g2s(&cl_s[0], cl_g + (size_t)cb0 * CREC, ns * CREC * 8u, &bar_c);
    };
    if (threadIdx.x == 0) {
        mbar_init(&bar[0], 1);
        mbar_init(&bar[1], 1);
        mbar_init(&bar_c, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    unsigned it = 0, tile = blockIdx.x;   // (the grid never exceeds the tiles)
    if (threadIdx.x == 0) {
        post_links(tile, 0);
        if (CLOV) post_clover(tile);
    }
    do {
        const int buf = it & 1;
        const unsigned par = (it >> 1) & 1, cpar = it & 1;
        if (threadIdx.x == 0) {   // draw the next tile and post its links; buf^1 was released by the barrier that ended iteration it-1
            const unsigned nt = gridDim.x + atomicAdd(&sched[0], 1u);
            next_s[buf] = nt;
            if (nt < ntiles) post_links(nt, buf ^ 1);
        }
        const unsigned j = tile * 32u + threadIdx.x;
        const bool active = j < (unsigned)g.Vh * B;
        const int cb = j / B, rhs = j % B;
        const int site = cb - tile * SITES;
        cx<double> acc[12];
        double d0 = 0.0;
        if (active) {
            const Coord c = decode(g, cb, p);
            HopAcc<double> hacc;
            hacc.zero();
            {   // forward-t frontier into L2 (dslash3_kernel.cuh): lane (site, rhs) takes rows rhs, rhs + 8 of its site's neighbour line set
                bool wrap;
                const int nbt = neighbour<3, 1>(g, cb, c, wrap);
                const double2 *q2 = a.in + lb_index((unsigned)nbt * B, 0, 12);
                prefetch_l2(q2 + 32 * rhs);
                if (rhs < 4) prefetch_l2(q2 + 32 * (rhs + 8));
            }
            const double *rec = &lk_s[buf][site * LREC];
            HopIn<double> d;
#define CLV_GAT3D(MU, FW) { bool wrap; const int nb = neighbour<MU, FW>(g, cb, c, wrap); load_spinor(a.in, (unsigned)nb * B + rhs, d.psi); d.neg = wrap && g.bc[MU] < 0; }
#define CLV_HOP3D(MU, FW) lds_link64<2 * MU + 1 - FW>(rec, d.u); hop_compute<double, 18, MU, FW>(d, hacc);
            CLV_GAT3D(0, 1)
            mbar_wait(&bar[buf], par);   // this tile's links have landed (posted one tile ahead)
            CLV_HOP3D(0, 1) CLV_GAT3D(0, 0) CLV_HOP3D(0, 0) CLV_GAT3D(1, 1) CLV_HOP3D(1, 1) CLV_GAT3D(1, 0) CLV_HOP3D(1, 0)
            CLV_GAT3D(2, 1) CLV_HOP3D(2, 1) CLV_GAT3D(2, 0) CLV_HOP3D(2, 0) CLV_GAT3D(3, 1) CLV_HOP3D(3, 1) CLV_GAT3D(3, 0) CLV_HOP3D(3, 0)
#undef CLV_GAT3D
#undef CLV_HOP3D
            hacc.finish(acc);
#pragma unroll
            for (int i = 0; i < 12; i++) acc[i] = a.coef * acc[i];
            cx<double> x[12];
            if (XMODE != XM_NONE) load_spinor(a.xin, j, x);
            if (XMODE == XM_PLAIN) {
#pragma unroll
                for (int i = 0; i < 12; i++) acc[i] = acc[i] + x[i];
            }
            if (CLOV) {
                mbar_wait(&bar_c, cpar);
                const double2 *srow = reinterpret_cast<const double2 *>(&cl_s[site * CREC]);
                if (XMODE == XM_CLOVER) clover_mul_rows<true>(srow, x, acc);
                if (PINV) {
                    cx<double> t[12];
                    clover_mul_rows<false>(srow, acc, t);
#pragma unroll
                    for (int i = 0; i < 12; i++) acc[i] = t[i];
                }
            }
        } else {
            mbar_wait(&bar[buf], par);
            if (CLOV) mbar_wait(&bar_c, cpar);
        }
        if (CLOV) {   // the clover buffer has been read: it takes the next tile's blocks while this tile is finished and the next one hops
            __syncthreads();
            if (threadIdx.x == 0 && next_s[buf] < ntiles) post_clover(next_s[buf]);
        }
        if (active) {
            if (DOT == DOT_RES) {  // residual epilogue: result = w - acc, ||result||^2, stored in the iteration precision (or not at all)
                cx<double> w[12];
                load_spinor(a.w, j, w);
#pragma unroll
                for (int i = 0; i < 12; i++) {
                    acc[i] = w[i] - acc[i];
                    d0 += acc[i].re * acc[i].re + acc[i].im * acc[i].im;
                }
                if (a.out32) {
                    cx<float> f[12];
#pragma unroll
                    for (int i = 0; i < 12; i++) f[i] = mk<float>((float)acc[i].re, (float)acc[i].im);
                    store_spinor(a.out32, j, f);
                } else if (a.out) store_spinor(a.out, j, acc);   // neither: only the norm is wanted (final verification)
            } else store_spinor(a.out, j, acc);
        }
        if (DOT == DOT_RES) {   // sum over the tile's 4 sites (lane bits 3, 4); one line of partial sums per TILE, indexed by the tile, so that
            // the scalar kernel's fixed-order sum does not depend on the scheduler (bit-reproducible)
            d0 += __shfl_xor_sync(0xffffffffu, d0, 8);
            d0 += __shfl_xor_sync(0xffffffffu, d0, 16);
            if (threadIdx.x < B) {
                double *o = a.partial + ((size_t)tile * B + threadIdx.x) * 4;
                o[0] = d0;
                o[1] = o[2] = o[3] = 0.0;
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
