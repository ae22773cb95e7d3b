// api.cu -- the extern "C" boundary declared in include/clover.h: argument checks and dispatch only.
#include "context.h"
#include <new>

namespace clv {
const char *last_error();
}
using namespace clv;

static int check_dims(const int dims[4])
{
    if (!dims) { set_error("dims is null"); return CLOVER_EINVAL; }
    long long V = 1;
    for (int m = 0; m < 4; m++) {
        if (dims[m] < 2 || (dims[m] & 1)) { set_error("extent %d of direction %d must be even and >= 2", dims[m], m); return CLOVER_EINVAL; }
        V *= dims[m];
    }
    if (V * 8 * 12 >= (1LL << 31)) { set_error("lattice too large for 32-bit vector indices (V = %lld)", V); return CLOVER_EINVAL; }
    return 0;
}

static int check_device()
{
    int n = 0;
    cudaError_t e = cudaGetDeviceCount(&n);
    if (e != cudaSuccess || n == 0) {
        set_error("no CUDA device: %s (this library has no CPU fallback)", e != cudaSuccess ? cudaGetErrorString(e) : "device count is 0");
        return CLOVER_ECUDA;
    }
    return 0;
}

extern "C" {

int clover_create(clover_ctx **out, const double *gauge_dev, const int dims[4], double kappa, double c_sw, const int bc[4], const clover_opts *opts,
                  void *stream)
{
    if (!out || !gauge_dev || !bc) { set_error("clover_create: null argument"); return CLOVER_EINVAL; }
    *out = nullptr;
    CLV_CHECK(check_dims(dims));
    for (int m = 0; m < 4; m++)
        if (bc[m] != 1 && bc[m] != -1) { set_error("bc[%d] = %d must be +1 or -1", m, bc[m]); return CLOVER_EINVAL; }
    const int recon = opts ? opts->recon : 18, max_rhs = opts ? opts->max_rhs : 8;
    if (recon != 18 && recon != 12) { set_error("recon = %d: supported values are 18 and 12", recon); return CLOVER_EINVAL; }
    if (max_rhs < 1 || max_rhs > 8) { set_error("max_rhs = %d must be in 1..8", max_rhs); return CLOVER_EINVAL; }
    CLV_CHECK(check_device());
    clover_ctx *ctx = new (std::nothrow) clover_ctx();
    if (!ctx) { set_error("out of host memory"); return CLOVER_ENOMEM; }
    Geom &g = ctx->geom;
    g.X = dims[0]; g.Y = dims[1]; g.Z = dims[2]; g.T = dims[3];
    g.Xh = g.X / 2;
    g.Vh = g.X * g.Y * g.Z * g.T / 2;
    for (int m = 0; m < 4; m++) g.bc[m] = bc[m];
    ctx->kappa = kappa;
    ctx->csw = c_sw;
    ctx->max_rhs = max_rhs;
    ctx->op64.recon = 18;
    ctx->op32.recon = recon;
    ctx->work = nullptr;
    const int rc = setup_operator(ctx, gauge_dev, (cudaStream_t)stream);
    if (rc < 0) { clover_destroy(ctx); return rc; }
    *out = ctx;
    return 0;
}

void clover_destroy(clover_ctx *ctx)
{
    if (!ctx) return;
    free_work(ctx);
    for (void *p : ctx->allocs) cudaFree(p);
    delete ctx;
}

int dslash_apply(clover_ctx *ctx, int op, int precision, const void *in_dev, void *out_dev, int n_rhs, void *stream)
{
    if (!ctx || !in_dev || !out_dev) { set_error("dslash_apply: null argument"); return CLOVER_EINVAL; }
    if (in_dev == out_dev) { set_error("dslash_apply: in and out must not alias"); return CLOVER_EINVAL; }
    if (precision != 32 && precision != 64) { set_error("precision = %d must be 32 or 64", precision); return CLOVER_EINVAL; }
    if (n_rhs < 0) { set_error("n_rhs = %d is negative", n_rhs); return CLOVER_EINVAL; }
    if (op < CLOVER_OP_HOP_EO || op > CLOVER_OP_MHAT) { set_error("dslash_apply: unknown op %d", op); return CLOVER_EINVAL; }
    if (n_rhs == 0) return 0;
    return apply_op(ctx, op, precision, in_dev, out_dev, n_rhs, (cudaStream_t)stream);
}

static int solve_common(clover_ctx *ctx, const double *src, double *dst, int n_rhs, double tol, int max_iter, int batch, int mixed,
                        clover_rhs_info *info, void *stream, int host)
{
    if (!ctx || !src || !dst || !info) { set_error("clover_solve: null argument"); return CLOVER_EINVAL; }
    if (n_rhs < 0) { set_error("n_rhs = %d is negative", n_rhs); return CLOVER_EINVAL; }
    if (batch != 1 && batch != 2 && batch != 4 && batch != 8) { set_error("batch = %d must be 1, 2, 4 or 8", batch); return CLOVER_EINVAL; }
    if (batch > ctx->max_rhs) { set_error("batch = %d exceeds max_rhs = %d", batch, ctx->max_rhs); return CLOVER_EINVAL; }
    if (!(tol > 0.0)) { set_error("tol must be positive"); return CLOVER_EINVAL; }
    if (max_iter < 1) { set_error("max_iter must be >= 1"); return CLOVER_EINVAL; }
    if (n_rhs == 0) return 0;
    return solve_batches(ctx, src, dst, n_rhs, tol, max_iter, batch, mixed != 0, info, (cudaStream_t)stream, host);
}

int clover_solve(clover_ctx *ctx, const double *sources_dev, double *propagators_dev, int n_rhs, double tol, int max_iter, int batch, int mixed,
                 clover_rhs_info *info_host, void *stream)
{
    return solve_common(ctx, sources_dev, propagators_dev, n_rhs, tol, max_iter, batch, mixed, info_host, stream, 0);
}

int clover_solve_host(clover_ctx *ctx, const double *sources_host, double *propagators_host, int n_rhs, double tol, int max_iter, int batch, int mixed,
                      clover_rhs_info *info_host, void *stream)
{
    return solve_common(ctx, sources_host, propagators_host, n_rhs, tol, max_iter, batch, mixed, info_host, stream, 1);
}

int noise_fill(void *out_dev, int precision, const int dims[4], uint64_t seed, int n_rhs, int rhs_offset, int dilution, double scale, void *stream)
{
    if (!out_dev) { set_error("noise_fill: null output"); return CLOVER_EINVAL; }
    CLV_CHECK(check_dims(dims));
    if (precision != 32 && precision != 64) { set_error("precision = %d must be 32 or 64", precision); return CLOVER_EINVAL; }
    if (n_rhs < 0 || rhs_offset < 0) { set_error("noise_fill: negative n_rhs or rhs_offset"); return CLOVER_EINVAL; }
    CLV_CHECK(check_device());
    if (dilution < 0 || dilution > 3) { set_error("noise_fill: dilution = %d must be 0..3 (bit 0 time, bit 1 spin-colour)", dilution); return CLOVER_EINVAL; }
    return launch_noise(out_dev, precision, dims, seed, n_rhs, rhs_offset, dilution, scale, (cudaStream_t)stream);
}

int stochastic_operators(const double *eta_dev, const double *x_dev, const int dims[4], int n_rhs, double *o_dev, void *stream)
{
    if (!eta_dev || !x_dev || !o_dev) { set_error("stochastic_operators: null argument"); return CLOVER_EINVAL; }
    CLV_CHECK(check_dims(dims));
    if (n_rhs < 1) { set_error("stochastic_operators: n_rhs = %d must be >= 1", n_rhs); return CLOVER_EINVAL; }
    CLV_CHECK(check_device());
    return launch_contract(eta_dev, x_dev, dims, n_rhs, o_dev, (cudaStream_t)stream);
}

int stochastic_operators_noalloc(const double *eta_dev, const double *x_dev, const int dims[4], int n_rhs, double *o_dev, void *stream)
{
    if (!eta_dev || !x_dev || !o_dev) { set_error("stochastic_operators_noalloc: null argument"); return CLOVER_EINVAL; }
    CLV_CHECK(check_dims(dims));
    if (n_rhs < 1) { set_error("stochastic_operators_noalloc: n_rhs = %d must be >= 1", n_rhs); return CLOVER_EINVAL; }
    if ((long long)dims[3] * n_rhs * n_rhs > CLOVER_NOALLOC_MAX_TNN) {
        set_error("stochastic_operators_noalloc: T * n_rhs^2 = %lld exceeds CLOVER_NOALLOC_MAX_TNN = %d (use stochastic_operators)",
                  (long long)dims[3] * n_rhs * n_rhs, CLOVER_NOALLOC_MAX_TNN);
        return CLOVER_EINVAL;
    }
    CLV_CHECK(check_device());
    return launch_contract_noalloc(eta_dev, x_dev, dims, n_rhs, o_dev, (cudaStream_t)stream);
}

int stochastic_correlator(const double *o_dev, int T, int n_rhs, double scale, double *c_dev, void *stream)
{
    if (!o_dev || !c_dev) { set_error("stochastic_correlator: null argument"); return CLOVER_EINVAL; }
    if (T < 1 || n_rhs < 1 || !(scale > 0.0)) { set_error("stochastic_correlator: bad T, n_rhs or scale"); return CLOVER_EINVAL; }
    CLV_CHECK(check_device());
    return launch_correlator(o_dev, T, n_rhs, scale, c_dev, (cudaStream_t)stream);
}

int stochastic_fill(const double *x_dev, const double *eta_dev, const int dims[4], int n_rhs, int t0, double scale, int dagger, double *s_dev,
                    void *stream)
{
    if (!x_dev || !eta_dev || !s_dev) { set_error("stochastic_fill: null argument"); return CLOVER_EINVAL; }
    CLV_CHECK(check_dims(dims));
    if (n_rhs < 1 || t0 < 0 || t0 >= dims[3] || !(scale > 0.0)) { set_error("stochastic_fill: bad n_rhs, t0 or scale"); return CLOVER_EINVAL; }
    const long long rows = 12LL * dims[0] * dims[1] * dims[2] * dims[3];
    if (rows / 64 + 1 > 65535) { set_error("stochastic_fill: lattice too large (the 12V x 12L^3 array would not fit any GPU)"); return CLOVER_EINVAL; }
    CLV_CHECK(check_device());
    return launch_fill(x_dev, eta_dev, dims, n_rhs, t0, scale, dagger != 0, s_dev, (cudaStream_t)stream);
}

int timeslice_norm2(const double *f_dev, long long n_outer, int T, long long slice_len, double *out_dev, void *stream)
{
    if (!f_dev || !out_dev) { set_error("timeslice_norm2: null argument"); return CLOVER_EINVAL; }
    if (n_outer < 1 || T < 1 || T > 65535 || slice_len < 1) { set_error("timeslice_norm2: bad n_outer, T or slice_len"); return CLOVER_EINVAL; }
    CLV_CHECK(check_device());
    return launch_timeslice_norm2(f_dev, (long)n_outer, T, (long)slice_len, out_dev, (cudaStream_t)stream);
}

int timeslice_inner(const double *a_dev, const double *b_dev, long long n_outer, int T, long long slice_len, double *out_dev, void *stream)
{
    if (!a_dev || !b_dev || !out_dev) { set_error("timeslice_inner: null argument"); return CLOVER_EINVAL; }
    if (n_outer < 1 || T < 1 || T > 65535 || slice_len < 1) { set_error("timeslice_inner: bad n_outer, T or slice_len"); return CLOVER_EINVAL; }
    CLV_CHECK(check_device());
    return launch_timeslice_inner(a_dev, b_dev, (long)n_outer, T, (long)slice_len, out_dev, (cudaStream_t)stream);
}

int clover_bench_kernel(clover_ctx *ctx, int kernel, int precision, int n_rhs, int reps, int flush_l2, float *ms_per_launch, void *stream)
{
    if (!ctx || !ms_per_launch) { set_error("clover_bench_kernel: null argument"); return CLOVER_EINVAL; }
    if (precision != 32 && precision != 64) { set_error("precision = %d must be 32 or 64", precision); return CLOVER_EINVAL; }
    if (n_rhs != 1 && n_rhs != 2 && n_rhs != 4 && n_rhs != 8) { set_error("n_rhs = %d must be 1, 2, 4 or 8", n_rhs); return CLOVER_EINVAL; }
    if (n_rhs > ctx->max_rhs) { set_error("n_rhs = %d exceeds max_rhs = %d", n_rhs, ctx->max_rhs); return CLOVER_EINVAL; }
    if (reps < 1) { set_error("reps must be >= 1"); return CLOVER_EINVAL; }
    return bench_kernel(ctx, kernel, precision, n_rhs, reps, flush_l2, ms_per_launch, (cudaStream_t)stream);
}

int clover_get_stats(const clover_ctx *ctx, clover_solve_stats *out)
{
    if (!ctx || !out) { set_error("clover_get_stats: null argument"); return CLOVER_EINVAL; }
    *out = ctx->stats;
    return 0;
}

const char *clover_last_error(const clover_ctx *) { return clv::last_error(); }

}  // extern "C"
