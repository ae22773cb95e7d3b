// dslash_inst.cuh -- host dispatch of one (precision, batch) family of Dslash kernels; included by the
// dslash_<prec>_b<B>.cu instantiation units so the variants compile in parallel.
#pragma once
#include "dslash3_kernel.cuh"
#ifdef CLV_BUILD_DSLASH3D   // defined by dslash_f64_b8.cu only: the fp64 B = 8 kernels are built once
#include "dslash3d_kernel.cuh"
#endif
#include <algorithm>
#include <cstdlib>

namespace clv {

// variants with a per-CTA reduction keep DSLASH_BLOCK threads; the others (DOT_NONE, DOT_S) run one-warp CTAs
#define CLV_HAS_RED(DT) ((DT) != DOT_NONE && (DT) != DOT_S)

// fp32, B >= 2: the (site, rhs-pair) kernel of dslash2_kernel.cuh
template <int B, int RECON>
static int launch_dslash2_BR(const clover_ctx *ctx, const OpData<float> &op, const DslashArgs<float> &a, cudaStream_t st, int *grid_out)
{
    const Geom &g = ctx->geom;
    const unsigned npairs = (unsigned)g.Vh * B / 2;
    const unsigned block = CLV_HAS_RED(a.dot) ? CLV_R2_BLOCK_DOT : CLV_R2_BLOCK_NODOT;
    const unsigned grid = (npairs + block - 1) / block;
    if (grid_out) *grid_out = (int)grid;
    const int key = a.xmode * 100 + a.pinv * 10 + a.dot;
#define CLV_LAUNCH2(XM, PI, DT)                                                      \
    case (XM) * 100 + (PI) * 10 + (DT):                                              \
        dslash2_kernel<B, RECON, XM, PI, DT, (CLV_HAS_RED(DT) ? CLV_R2_BLOCK_DOT : CLV_R2_BLOCK_NODOT)><<<grid, block, 0, st>>>(g, op, a); \
        break;
    switch (key) {
        CLV_LAUNCH2(XM_NONE, 0, DOT_NONE)
        CLV_LAUNCH2(XM_NONE, 1, DOT_NONE)
        CLV_LAUNCH2(XM_PLAIN, 0, DOT_NONE)
        CLV_LAUNCH2(XM_PLAIN, 1, DOT_NONE)
        CLV_LAUNCH2(XM_CLOVER, 0, DOT_NONE)
        CLV_LAUNCH2(XM_CLOVER, 0, DOT_W)
        CLV_LAUNCH2(XM_CLOVER, 0, DOT_X)
        CLV_LAUNCH2(XM_CLOVER, 0, DOT_RES)
        CLV_LAUNCH2(XM_CLOVER, 0, DOT_S)
        CLV_LAUNCH2(XM_CLOVER, 0, DOT_XW)
    default:
        set_error("dslash: unsupported variant xmode=%d pinv=%d dot=%d", a.xmode, a.pinv, a.dot);
        return CLOVER_EINVAL;
    }
#undef CLV_LAUNCH2
    CLV_CUDA(cudaGetLastError());
    return 0;
}
// fp32, B = 8: the persistent kernel of dslash3_kernel.cuh (operator data by bulk async copy): grid = the one-warp CTAs resident on the
// device.  The shared-memory carveout is set to what the resident CTAs need (+1 KB per CTA the system reserves) so that the rest of the
// SM's 228 KB stays L1 for the gathers.
#ifndef CLV_R3_GRID_PER_SM
#define CLV_R3_GRID_PER_SM 12   // persistent one-warp CTAs launched per SM (<= the resident limit of the launch bounds)
#endif
// smallest shared-memory carveout of sm_100 (KB) that holds `ctas` CTAs of `bytes` static shared memory + 1 KB each, as a percentage of 228 KB
static int r3_carveout_pct(size_t bytes, int ctas)
{
    static const int kb[] = {8, 16, 32, 64, 100, 132, 164, 196, 228};
    const size_t need = (bytes + 1024) * ctas;
    for (int k : kb)
        if ((size_t)k * 1024 >= need) return (k * 100 + 227) / 228;
    return 100;
}
template <int B, int RECON>
static int launch_dslash3_BR(const clover_ctx *ctx, const OpData<float> &op, const DslashArgs<float> &a, cudaStream_t st, int *grid_out)
{
    const Geom &g = ctx->geom;
    static const int n_sm = [] { int dev = 0, n = 148; cudaGetDevice(&dev); cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev); return n; }();
    const int key = a.xmode * 100 + a.pinv * 10 + a.dot;
#define CLV_LAUNCH3(XM, PI, DT)                                                                                          \
    case (XM) * 100 + (PI) * 10 + (DT): {                                                                                \
        constexpr int BLK = 32;                                                                                          \
        auto kern = dslash3_kernel<B, RECON, XM, PI, DT, BLK>;                                                           \
        static const cudaError_t attr = [&] {                                                                            \
            cudaFuncAttributes fa;                                                                                       \
            cudaError_t e = cudaFuncGetAttributes(&fa, kern);                                                            \
            if (e != cudaSuccess) return e;                                                                              \
            e = cudaFuncSetAttribute(kern, cudaFuncAttributePreferredSharedMemoryCarveout, r3_carveout_pct(fa.sharedSizeBytes, CLV_R3_GRID_PER_SM)); \
            return e;                                                                                                    \
        }();                                                                                                             \
        CLV_CUDA(attr);                                                                                                  \
        const unsigned ntiles = ((unsigned)g.Vh + (2 * BLK / B) - 1) / (2 * BLK / B);                                    \
        const unsigned grid = std::min<unsigned>(ntiles, (unsigned)n_sm * CLV_R3_GRID_PER_SM);                           \
        if (grid_out) *grid_out = (int)ntiles;   /* lines of partial sums: one per tile */                                \
        kern<<<grid, BLK, 0, st>>>(g, op, a, ctx->sched);                                                                \
        break;                                                                                                           \
    }
    switch (key) {
        CLV_LAUNCH3(XM_NONE, 0, DOT_NONE)
        CLV_LAUNCH3(XM_NONE, 1, DOT_NONE)
        CLV_LAUNCH3(XM_PLAIN, 0, DOT_NONE)
        CLV_LAUNCH3(XM_PLAIN, 1, DOT_NONE)
        CLV_LAUNCH3(XM_CLOVER, 0, DOT_NONE)
        CLV_LAUNCH3(XM_CLOVER, 0, DOT_W)
        CLV_LAUNCH3(XM_CLOVER, 0, DOT_X)
        CLV_LAUNCH3(XM_CLOVER, 0, DOT_RES)
        CLV_LAUNCH3(XM_CLOVER, 0, DOT_S)
        CLV_LAUNCH3(XM_CLOVER, 0, DOT_XW)
    default:
        set_error("dslash: unsupported variant xmode=%d pinv=%d dot=%d", a.xmode, a.pinv, a.dot);
        return CLOVER_EINVAL;
    }
#undef CLV_LAUNCH3
    CLV_CUDA(cudaGetLastError());
    return 0;
}

#ifdef CLV_BUILD_DSLASH3D
// fp64, B = 8, the variants of the mixed-precision solve: dslash3d_kernel.cuh (persistent, one thread per site and rhs); false if not built
static bool launch_dslash3d(const clover_ctx *ctx, const OpData<double> &op, const DslashArgs<double> &a, cudaStream_t st, int *grid_out, int *rc)
{
    const Geom &g = ctx->geom;
    static const int n_sm = [] { int dev = 0, n = 148; cudaGetDevice(&dev); cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev); return n; }();
    const int key = a.xmode * 100 + a.pinv * 10 + a.dot;
    *rc = 0;
#define CLV_LAUNCH3D(XM, PI, DT)                                                                                         \
    case (XM) * 100 + (PI) * 10 + (DT): {                                                                                \
        auto kern = dslash3d_kernel<XM, PI, DT>;                                                                         \
        static const cudaError_t attr = [&] {                                                                            \
            cudaFuncAttributes fa;                                                                                       \
            cudaError_t e = cudaFuncGetAttributes(&fa, kern);                                                            \
            if (e != cudaSuccess) return e;                                                                              \
            return cudaFuncSetAttribute(kern, cudaFuncAttributePreferredSharedMemoryCarveout, r3_carveout_pct(fa.sharedSizeBytes, CLV_R3D_WARPS_PER_SM)); \
        }();                                                                                                             \
        if (attr != cudaSuccess) { set_error("cudaFuncSetAttribute failed: %s", cudaGetErrorString(attr)); *rc = CLOVER_ECUDA; return true; } \
        const unsigned ntiles = ((unsigned)g.Vh + 3) / 4;                                                                \
        const unsigned grid = std::min<unsigned>(ntiles, (unsigned)n_sm * CLV_R3D_WARPS_PER_SM);                         \
        if (grid_out) *grid_out = (int)ntiles;   /* lines of partial sums: one per tile */                                \
        kern<<<grid, 32, 0, st>>>(g, op, a, ctx->sched);                                                                 \
        break;                                                                                                           \
    }
    switch (key) {
        CLV_LAUNCH3D(XM_NONE, 1, DOT_NONE)
        CLV_LAUNCH3D(XM_PLAIN, 0, DOT_NONE)
        CLV_LAUNCH3D(XM_PLAIN, 1, DOT_NONE)
        CLV_LAUNCH3D(XM_CLOVER, 0, DOT_RES)
    default: return false;
    }
#undef CLV_LAUNCH3D
    if (cudaGetLastError() != cudaSuccess) { set_error("dslash3d launch failed"); *rc = CLOVER_ECUDA; }
    return true;
}
#endif
template <typename R, int B> struct Launch3D {
    static bool go(const clover_ctx *, const OpData<R> &, const DslashArgs<R> &, cudaStream_t, int *, int *) { return false; }
};
#ifdef CLV_BUILD_DSLASH3D
template <> struct Launch3D<double, 8> {
    static bool go(const clover_ctx *ctx, const OpData<double> &op, const DslashArgs<double> &a, cudaStream_t st, int *grid_out, int *rc)
    {
        static const bool on = [] { const char *e = getenv("CLOVER_R3D"); return e ? atoi(e) != 0 : true; }();  // tuning/debug knob only
        return on && launch_dslash3d(ctx, op, a, st, grid_out, rc);
    }
};
#endif

template <typename R, int B, int RECON> struct PairLaunch {   // double, or B = 1: no pair kernel
    static bool use() { return false; }
    static int go(const clover_ctx *, const OpData<R> &, const DslashArgs<R> &, cudaStream_t, int *) { return CLOVER_EINVAL; }
};
template <int B, int RECON> struct PairLaunchF {
    static bool use()
    {
        static const bool on = [] { const char *e = getenv("CLOVER_R2"); return e ? atoi(e) != 0 : true; }();  // tuning/debug knob only
        return on;
    }
    static int go(const clover_ctx *ctx, const OpData<float> &op, const DslashArgs<float> &a, cudaStream_t st, int *grid_out)
    {
        return launch_dslash2_BR<B, RECON>(ctx, op, a, st, grid_out);
    }
};
template <int RECON> struct PairLaunch<float, 2, RECON> : PairLaunchF<2, RECON> {};
template <int RECON> struct PairLaunch<float, 4, RECON> : PairLaunchF<4, RECON> {};
template <int RECON> struct PairLaunch<float, 8, RECON> : PairLaunchF<8, RECON> {
    static int go(const clover_ctx *ctx, const OpData<float> &op, const DslashArgs<float> &a, cudaStream_t st, int *grid_out)
    {
        static const bool r3 = [] { const char *e = getenv("CLOVER_R3"); return e ? atoi(e) != 0 : true; }();  // tuning/debug knob only
        return r3 ? launch_dslash3_BR<8, RECON>(ctx, op, a, st, grid_out) : launch_dslash2_BR<8, RECON>(ctx, op, a, st, grid_out);
    }
};


template <typename R, int B, int RECON>
static int launch_dslash_BR(const clover_ctx *ctx, const OpData<R> &op, const DslashArgs<R> &a, cudaStream_t st, int *grid_out)
{
    // B = 2, 4: the pair kernel wins where link AND clover loads are shared (the fused solver kernels), the plain hop stays per-rhs;
    // B = 8: the persistent kernel takes every variant (plain hop at 24^3x48: 149 us against 191 us per-rhs)
    if (PairLaunch<R, B, RECON>::use() && (a.xmode != XM_NONE || a.pinv || B == 8)) return PairLaunch<R, B, RECON>::go(ctx, op, a, st, grid_out);
    {
        int rc3 = 0;
        if (Launch3D<R, B>::go(ctx, op, a, st, grid_out, &rc3)) return rc3;
    }
    const Geom &g = ctx->geom;
    const unsigned n = (unsigned)g.Vh * B;
    const unsigned block = CLV_HAS_RED(a.dot) ? DSLASH_BLOCK : CLV_DSLASH_BLOCK_NODOT;
    const unsigned grid = (n + block - 1) / block;
    if (grid_out) *grid_out = (int)grid;
    const int key = a.xmode * 100 + a.pinv * 10 + a.dot;
#define CLV_LAUNCH(XM, PI, DT)                                                          \
    case (XM) * 100 + (PI) * 10 + (DT):                                                 \
        dslash_kernel<R, B, RECON, XM, PI, DT, (CLV_HAS_RED(DT) ? DSLASH_BLOCK : CLV_DSLASH_BLOCK_NODOT)><<<grid, block, 0, st>>>(g, op, a); \
        break;
    switch (key) {
        CLV_LAUNCH(XM_NONE, 0, DOT_NONE)
        CLV_LAUNCH(XM_NONE, 1, DOT_NONE)
        CLV_LAUNCH(XM_PLAIN, 0, DOT_NONE)
        CLV_LAUNCH(XM_PLAIN, 1, DOT_NONE)
        CLV_LAUNCH(XM_CLOVER, 0, DOT_NONE)
        CLV_LAUNCH(XM_CLOVER, 0, DOT_W)
        CLV_LAUNCH(XM_CLOVER, 0, DOT_X)
        CLV_LAUNCH(XM_CLOVER, 0, DOT_RES)
        CLV_LAUNCH(XM_CLOVER, 0, DOT_S)
        CLV_LAUNCH(XM_CLOVER, 0, DOT_XW)
    default:
        set_error("dslash: unsupported variant xmode=%d pinv=%d dot=%d", a.xmode, a.pinv, a.dot);
        return CLOVER_EINVAL;
    }
#undef CLV_LAUNCH
    CLV_CUDA(cudaGetLastError());
    return 0;
}

template <typename R> struct OpSel;
template <> struct OpSel<float> { static const OpData<float> &get(const clover_ctx *c) { return c->op32; } };
template <> struct OpSel<double> { static const OpData<double> &get(const clover_ctx *c) { return c->op64; } };

template <typename R, int B> int launch_dslash_B(const clover_ctx *ctx, const DslashArgs<R> &a, cudaStream_t st, int *grid_out)
{
    const OpData<R> &op = OpSel<R>::get(ctx);
    if (op.recon == 12) {
        if (sizeof(R) == 4) return launch_dslash_BR<R, B, (sizeof(R) == 4 ? 12 : 18)>(ctx, op, a, st, grid_out);
        set_error("dslash: two-row links exist in fp32 only");
        return CLOVER_EINVAL;
    }
    return launch_dslash_BR<R, B, 18>(ctx, op, a, st, grid_out);
}

template <typename R, int B>
int launch_clover_B(const clover_ctx *ctx, const typename Vec<R>::T *in, typename Vec<R>::T *out, int parity, int inverse, cudaStream_t st)
{
    const Geom &g = ctx->geom;
    const OpData<R> &op = OpSel<R>::get(ctx);
    const unsigned n = (unsigned)g.Vh * B;
    clover_kernel<R, B><<<(n + DSLASH_BLOCK - 1) / DSLASH_BLOCK, DSLASH_BLOCK, 0, st>>>(g, inverse ? op.clov_inv[parity] : op.clov[parity], in, out);
    CLV_CUDA(cudaGetLastError());
    return 0;
}

}  // namespace clv
