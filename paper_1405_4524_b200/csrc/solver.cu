// solver.cu -- host driver of the batched, even-odd preconditioned, mixed-precision BiCGStab (
// 8(c) O6'): B independent recurrences share every operator application; all scalars stay on the device, the host
// only reads back the per-rhs flags once per iteration.
//   Mhat = A_ee - kappa^2 H_eo A_oo^-1 H_oe   on the even sites            (R13)
//   b_e  = eta_e + kappa H_eo A_oo^-1 eta_o ;  psi_o = A_oo^-1 (eta_o + kappa H_oe psi_e)
// Also: dslash_apply's operator table and the kernel benchmark entry.
#include "blas.cuh"
#include <algorithm>
#include <cmath>
#include <cstdlib>
#include <cstring>

namespace clv {

struct SolveWork {
    int B_cap = 0;
    size_t sloppy_bytes = 0;   // bytes of each sloppy field currently allocated
    double2 *f64[8] = {};      // eta_e, eta_o, b, y, r64, w64, tmp64, psi_o
    void *sl[9] = {};          // x, r, p, v, s, t, r0, tmp, q0  (float4 or double2 fields)
    double *partial = nullptr, *partial2 = nullptr;
    int partial_blocks = 0;
    double *stage = nullptr;
    unsigned *ticket = nullptr;
    RhsScalars *sc_dev = nullptr, *sc_host = nullptr;  // sc_host: mapped pinned memory the device writes the flags into
    RhsScalars *sc_host_dev = nullptr;                 // device address of sc_host
    // host-buffer solves: double-buffered canonical staging, copies on their own streams so that the H2D of batch i+1 and the
    // D2H of batch i-1 overlap the solve of batch i
    double *stage_in[2] = {}, *stage_out[2] = {};
    size_t stage_bytes = 0;
    cudaStream_t s_in = nullptr, s_out = nullptr;
    cudaEvent_t ev_in[2] = {}, ev_out[2] = {};
    void *flush = nullptr;
    cudaEvent_t ev[6] = {};
    cudaEvent_t kev[6] = {};   // per-launch timing of the two sloppy Mhat calls of an iteration: 2 x (start, mid, end)
    cudaEvent_t kev1[2][2] = {};   // merged iteration: start / end of its first Dslash, which is queued one iteration ahead (ping-pong)
    cudaEvent_t ev_flags = nullptr;   // merged iteration: the flags of the iteration are in host memory
    bool have_ev = false;
    // launch-bound lattices: one iteration (10 kernels + the flag read-back) replayed as a CUDA graph on an internal stream
    cudaStream_t s_work = nullptr;
    cudaEvent_t ev_dep = nullptr;
    cudaGraphExec_t iter_graph = nullptr;
    int graph_B = 0, graph_prec = 0, graph_kernels = 0, graph_merged = -1;
    double graph_tol2 = 0, graph_delta2 = 0;
};

enum { F_ETA_E = 0, F_ETA_O, F_B, F_Y, F_R64, F_W64, F_TMP64, F_PSI_O };
enum { S_X = 0, S_R, S_P, S_V, S_S, S_T, S_R0, S_TMP, S_Q0, S_NFIELDS };

void free_work(clover_ctx *ctx)
{
    SolveWork *W = ctx->work;
    if (!W) return;
    for (int i = 0; i < 8; i++) cudaFree(W->f64[i]);
    for (int i = 0; i < S_NFIELDS; i++) cudaFree(W->sl[i]);
    cudaFree(W->partial);
    cudaFree(W->partial2);
    cudaFree(W->stage);
    cudaFree(W->ticket);
    cudaFree(W->sc_dev);
    cudaFreeHost(W->sc_host);
    for (int k = 0; k < 2; k++) { cudaFree(W->stage_in[k]); cudaFree(W->stage_out[k]); if (W->ev_in[k]) cudaEventDestroy(W->ev_in[k]); if (W->ev_out[k]) cudaEventDestroy(W->ev_out[k]); }
    if (W->s_in) cudaStreamDestroy(W->s_in);
    if (W->s_out) cudaStreamDestroy(W->s_out);
    cudaFree(W->flush);
    if (W->have_ev) {
        for (int i = 0; i < 6; i++) { cudaEventDestroy(W->ev[i]); cudaEventDestroy(W->kev[i]); }
        for (int i = 0; i < 4; i++) cudaEventDestroy(W->kev1[i / 2][i % 2]);
        cudaEventDestroy(W->ev_flags);
    }
    if (W->iter_graph) cudaGraphExecDestroy(W->iter_graph);
    if (W->s_work) cudaStreamDestroy(W->s_work);
    if (W->ev_dep) cudaEventDestroy(W->ev_dep);
    delete W;
    ctx->work = nullptr;
}

// Workspaces are (re)allocated only when a call needs more than the context holds; their one-time clears are queued on the
// caller's stream, so a call that finds everything in place touches no other stream and never synchronises the device.
static int ensure_work(clover_ctx *ctx, int B, size_t real_bytes, bool staging, cudaStream_t st)
{
    if (!ctx->work) ctx->work = new SolveWork();
    SolveWork *W = ctx->work;
    const Geom &g = ctx->geom;
    if (B > W->B_cap) {
        const size_t n64 = field_vecs<double>(g, B);
        for (int i = 0; i < 8; i++) {
            cudaFree(W->f64[i]);
            W->f64[i] = nullptr;
            CLV_CUDA(cudaMalloc(&W->f64[i], n64 * sizeof(double2)));
            CLV_CUDA(cudaMemsetAsync(W->f64[i], 0, n64 * sizeof(double2), st));
        }
        cudaFree(W->partial);
        // twice the blocks of one Dslash launch: the final verification reduces the partials of two launches (even + odd) at once
        // (one line per 32 threads of a launch at most: the persistent B = 8 kernels write one line per tile of 8 or 4 sites)
        W->partial_blocks = 2 * std::max<int>(((unsigned)g.Vh * B + 31) / 32, 148 * 8);
        CLV_CUDA(cudaMalloc(&W->partial, (size_t)W->partial_blocks * B * 4 * sizeof(double)));
        CLV_CUDA(cudaMemsetAsync(W->partial, 0, (size_t)W->partial_blocks * B * 4 * sizeof(double), st));
        cudaFree(W->partial2);
        CLV_CUDA(cudaMalloc(&W->partial2, (size_t)W->partial_blocks * B * 4 * sizeof(double)));
        CLV_CUDA(cudaMemsetAsync(W->partial2, 0, (size_t)W->partial_blocks * B * 4 * sizeof(double), st));
        if (!W->sc_dev) {
            CLV_CUDA(cudaMalloc(&W->sc_dev, 8 * sizeof(RhsScalars)));
            CLV_CUDA(cudaMemsetAsync(W->sc_dev, 0, 8 * sizeof(RhsScalars), st));
            CLV_CUDA(cudaHostAlloc((void **)&W->sc_host, 8 * sizeof(RhsScalars), cudaHostAllocMapped));
            CLV_CUDA(cudaHostGetDevicePointer((void **)&W->sc_host_dev, W->sc_host, 0));
            CLV_CUDA(cudaMalloc(&W->stage, 8 * 32 * 8 * sizeof(double)));
            CLV_CUDA(cudaMalloc(&W->ticket, 8 * sizeof(unsigned)));
            CLV_CUDA(cudaMemsetAsync(W->ticket, 0, 8 * sizeof(unsigned), st));
        }
        W->B_cap = B;
        W->sloppy_bytes = 0;
        if (W->iter_graph) { cudaGraphExecDestroy(W->iter_graph); W->iter_graph = nullptr; }
    }
    const size_t need = field_vecs<double>(g, W->B_cap) * 16 / 8 * real_bytes;  // float fields are half the size of double ones
    if (need > W->sloppy_bytes) {
        for (int i = 0; i < S_NFIELDS; i++) {
            cudaFree(W->sl[i]);
            W->sl[i] = nullptr;
            CLV_CUDA(cudaMalloc(&W->sl[i], need));
            CLV_CUDA(cudaMemsetAsync(W->sl[i], 0, need, st));
        }
        W->sloppy_bytes = need;
        if (W->iter_graph) { cudaGraphExecDestroy(W->iter_graph); W->iter_graph = nullptr; }
    }
    if (staging) {
        const size_t sb = (size_t)2 * g.Vh * 24 * sizeof(double) * W->B_cap;
        if (sb > W->stage_bytes) {
            for (int k = 0; k < 2; k++) {
                cudaFree(W->stage_in[k]);
                cudaFree(W->stage_out[k]);
                W->stage_in[k] = W->stage_out[k] = nullptr;
                CLV_CUDA(cudaMalloc(&W->stage_in[k], sb));
                CLV_CUDA(cudaMalloc(&W->stage_out[k], sb));
            }
            W->stage_bytes = sb;
        }
        if (!W->s_in) {
            CLV_CUDA(cudaStreamCreateWithFlags(&W->s_in, cudaStreamNonBlocking));
            CLV_CUDA(cudaStreamCreateWithFlags(&W->s_out, cudaStreamNonBlocking));
            for (int k = 0; k < 2; k++) {
                CLV_CUDA(cudaEventCreateWithFlags(&W->ev_in[k], cudaEventDisableTiming));
                CLV_CUDA(cudaEventCreateWithFlags(&W->ev_out[k], cudaEventDisableTiming));
            }
        }
    }
    if (!W->have_ev) {
        for (int i = 0; i < 6; i++) { CLV_CUDA(cudaEventCreate(&W->ev[i])); CLV_CUDA(cudaEventCreate(&W->kev[i])); }
        for (int i = 0; i < 4; i++) CLV_CUDA(cudaEventCreate(&W->kev1[i / 2][i % 2]));
        CLV_CUDA(cudaEventCreateWithFlags(&W->ev_flags, cudaEventDisableTiming));
        CLV_CUDA(cudaStreamCreateWithFlags(&W->s_work, cudaStreamNonBlocking));
        CLV_CUDA(cudaEventCreateWithFlags(&W->ev_dep, cudaEventDisableTiming));
        W->have_ev = true;
    }
    return 0;
}

// Padding lanes (j >= Vh*B in the last 32-lane block) must hold zeros because the BLAS sweeps and their reductions
// run over whole blocks.  Only lattices with Vh*B not a multiple of 32 have any; there the fields are cleared
// whenever the batch size (hence the meaning of a lane) changes.
static int clear_fields(SolveWork *W, const Geom &g, int B, cudaStream_t st)
{
    if (((unsigned)g.Vh * B) % 32u == 0) return 0;
    const size_t n64 = field_vecs<double>(g, W->B_cap) * sizeof(double2);
    for (int i = 0; i < 8; i++) CLV_CUDA(cudaMemsetAsync(W->f64[i], 0, n64, st));
    for (int i = 0; i < S_NFIELDS; i++) CLV_CUDA(cudaMemsetAsync(W->sl[i], 0, W->sloppy_bytes, st));
    return 0;
}

template <typename R> static DslashArgs<R> dargs(const typename Vec<R>::T *in, const typename Vec<R>::T *xin, typename Vec<R>::T *out, R coef, int parity,
                                                int xmode, int pinv, int dot = DOT_NONE, const typename Vec<R>::T *w = nullptr, double *partial = nullptr)
{
    DslashArgs<R> a;
    a.in = in; a.xin = xin; a.out = out; a.w = w; a.out32 = nullptr; a.partial = partial; a.coef = coef; a.parity = parity;
    a.partial2 = nullptr; a.out2 = nullptr; a.sc = nullptr;
    a.xmode = xmode; a.pinv = pinv; a.dot = dot;
    return a;
}

// out_e = Mhat in_e, optional fused dot products; tmp is an odd-parity scratch field
template <typename R>
static int mhat(clover_ctx *ctx, int B, const typename Vec<R>::T *in, typename Vec<R>::T *tmp, typename Vec<R>::T *out, int dot, const typename Vec<R>::T *w,
                double *partial, int *grid, cudaStream_t st, cudaEvent_t *kev = nullptr, float4 *out32 = nullptr, typename Vec<R>::T *out2 = nullptr,
                double *partial2 = nullptr, const RhsScalars *sc = nullptr)
{
    const R k2 = (R)(-ctx->kappa * ctx->kappa);
    if (kev) CLV_CUDA(cudaEventRecord(kev[0], st));
    CLV_CHECK(launch_dslash<R>(ctx, dargs<R>(in, nullptr, tmp, (R)1, 1, XM_NONE, 1), B, st, nullptr));
    if (kev) CLV_CUDA(cudaEventRecord(kev[1], st));
    DslashArgs<R> a2 = dargs<R>(tmp, in, out, k2, 0, XM_CLOVER, 0, dot, w, partial);
    a2.out32 = out32;
    a2.out2 = out2;
    a2.partial2 = partial2;
    a2.sc = sc;
    CLV_CHECK(launch_dslash<R>(ctx, a2, B, st, grid));
    if (kev) CLV_CUDA(cudaEventRecord(kev[2], st));
    ctx->stats.kernel_launches += 2;
    return 0;
}

// Flag read-back: a 32-thread kernel stores the per-rhs scalars straight into mapped pinned host memory.  (A cudaMemcpyAsync
// would queue behind the gigabyte device-to-host copies of clover_solve_host on the copy engine and stall every iteration.)
__global__ void publish_scalars_kernel(const RhsScalars *__restrict__ src, RhsScalars *dst, int words)
{
    const unsigned long long *s = reinterpret_cast<const unsigned long long *>(src);
    volatile unsigned long long *d = reinterpret_cast<volatile unsigned long long *>(dst);
    for (int i = threadIdx.x; i < words; i += blockDim.x) d[i] = s[i];
    __threadfence_system();
}
static int publish_scalars(SolveWork *W, int B, cudaStream_t st)
{
    static_assert(sizeof(RhsScalars) % 8 == 0, "RhsScalars is copied in 8-byte words");
    publish_scalars_kernel<<<1, 32, 0, st>>>(W->sc_dev, W->sc_host_dev, B * (int)(sizeof(RhsScalars) / 8));
    CLV_CUDA(cudaGetLastError());
    return 0;
}
static int fetch_scalars(SolveWork *W, int B, cudaStream_t st)
{
    CLV_CHECK(publish_scalars(W, B, st));
    CLV_CUDA(cudaStreamSynchronize(st));
    return 0;
}

static double reliable_delta()
{
    const char *e = getenv("CLOVER_DELTA");  // tuning/debug knob only
    const double d = e ? atof(e) : 0.0;
    // 3e-6: two fp32 legs (1 -> 3e-6 -> 1e-10 relative to ||eta||), each well inside what fp32 recurrences resolve (the iterated
    // residual of a leg is good to ~1e-6 of the leg's start); measured at 24^3x48: 1e-4..1e-5 three fp64 recomputations per batch,
    // 3e-6 two with the same iteration count, 1e-6 two with one more iteration (profiles/r1_tuning.md)
    return (d > 0.0 && d < 1.0) ? d : 3e-6;
}

// Small lattices are launch-bound (a 16^3x32 Dslash takes ~10 us): replay the iteration as a CUDA graph there.
static bool graph_enabled(const Geom &g, int B)
{
    const char *e = getenv("CLOVER_GRAPH");  // tuning/debug knob only
    if (e) return atoi(e) != 0;
    return (size_t)g.Vh * B * 96 < ((size_t)64 << 20);
}

// The merged iteration (default) moves BLAS-1 traffic into the Dslash epilogues: alpha is known before Mhat p is applied
// (<r0, Mhat p> = <Mhat^+ r0, p>, Mhat^+ = gamma5 Mhat gamma5), so the second Dslash of Mhat p stores s = r - alpha v instead of v, the
// second Dslash of Mhat s also returns <r0,t> and <r0,s> (rho' = <r0,s> - omega <r0,t>), and one sweep does the x, r and p updates
// (p = r' + beta p - (rho'/rho)(r - s), since r - s = alpha v): 9 vector passes + 2 scalar steps per iteration instead of 14 + 3.  CLOVER_MERGED=0 selects the textbook ordering.
static bool merged_enabled()
{
    const char *e = getenv("CLOVER_MERGED");  // tuning/debug knob only
    return e ? atoi(e) != 0 : true;
}

template <typename R>
static int solve_batch(clover_ctx *ctx, const double *src, double *dst, int B, double tol, int max_iter, clover_rhs_info *info, cudaStream_t st_user)
{
    typedef typename Vec<R>::T V;
    SolveWork *W = ctx->work;
    const Geom &g = ctx->geom;
    const bool use_graph = graph_enabled(g, B);
    cudaStream_t st = st_user;
    if (use_graph) {  // the legacy default stream cannot be captured: run on the internal stream, ordered after the caller's work
        st = W->s_work;
        CLV_CUDA(cudaEventRecord(W->ev_dep, st_user));
        CLV_CUDA(cudaStreamWaitEvent(st, W->ev_dep, 0));
    }
    double2 *eta_e = W->f64[F_ETA_E], *eta_o = W->f64[F_ETA_O], *b = W->f64[F_B], *y = W->f64[F_Y],
            *tmp64 = W->f64[F_TMP64], *psi_o = W->f64[F_PSI_O];
    V *x = (V *)W->sl[S_X], *r = (V *)W->sl[S_R], *p = (V *)W->sl[S_P], *v = (V *)W->sl[S_V], *s = (V *)W->sl[S_S], *t = (V *)W->sl[S_T],
      *r0 = (V *)W->sl[S_R0], *tmp = (V *)W->sl[S_TMP], *q0 = (V *)W->sl[S_Q0];
    const bool merged = merged_enabled();
    long long &nl = ctx->stats.kernel_launches;
    // relative breakdown threshold of the recurrence (R11): 1e-10 in fp64 as in the oracle's spirit (it uses 1e-14; 1e-10 needs fewer iterations on
    // near-critical systems), 1e-6 for the fp32 iteration, whose dot products carry no more
    const double brk = sizeof(R) == 8 ? 1e-10 : 1e-6;
    BlasCtx bc{&g, B, W->sc_dev, W->partial, W->partial2, W->partial_blocks, W->stage, W->ticket, st, &nl, brk * brk};
    const double tol2 = tol * tol, delta = reliable_delta(), delta2 = delta * delta;
    const size_t nbytes = field_vecs<R>(g, B) * sizeof(V), nbytes64 = field_vecs<double>(g, B) * sizeof(double2);
    int nb = 0, grid = 0, iters = 0, updates = 0;
    float ms;

    CLV_CUDA(cudaEventRecord(W->ev[0], st));
    CLV_CHECK((reorder_in<double, double>(g, src, eta_e, eta_o, B, st)));
    nl++;
    CLV_CUDA(cudaEventRecord(W->ev[1], st));
    // stopping scale ||eta||^2 (R10) and source preparation b_e = eta_e + kappa H_eo A_oo^-1 eta_o
    CLV_CHECK(blas_norm2_pair(bc, eta_e, nullptr, eta_o, nullptr, &nb));
    CLV_CHECK(blas_scalar_step(bc, SC_ETA2, nb, tol2, delta2));
    CLV_CHECK(launch_clover<double>(ctx, eta_o, tmp64, 1, 1, B, st));
    CLV_CHECK(launch_dslash<double>(ctx, dargs<double>(tmp64, eta_e, b, ctx->kappa, 0, XM_PLAIN, 0), B, st, nullptr));
    nl += 2;
    // y = 0, x = 0, r = b, p = r0 = r
    CLV_CUDA(cudaMemsetAsync(y, 0, nbytes64, st));
    CLV_CUDA(cudaMemsetAsync(x, 0, nbytes, st));
    CLV_CHECK(blas_residual<R>(bc, b, nullptr, nullptr, r, &nb));   // r = (R) b, ||b||^2; no fp64 copy of r is kept
    CLV_CHECK(blas_scalar_step(bc, merged ? SC_INIT_MERGED : SC_INIT, nb, tol2, delta2));
    // merged iteration, (re)start of the rhs flagged `restart == 1`: r0 := p := r, q0 := Mhat^+ r0 = gamma5 Mhat gamma5 r0,
    // rho := ||r||^2, alpha := rho / <q0, p>.  s, t and tmp are free between iterations and serve as scratch.
    auto restart_merged = [&]() -> int {
        CLV_CHECK(blas_restart<R>(bc, r, r0, p));
        CLV_CHECK(blas_gamma5<R>(bc, r0, s, 0));
        CLV_CHECK(mhat<R>(ctx, B, s, tmp, t, DOT_NONE, nullptr, nullptr, nullptr, st));
        CLV_CHECK(blas_gamma5<R>(bc, t, q0, 1));
        CLV_CHECK(blas_cdot<R>(bc, q0, p, &nb));
        CLV_CHECK(blas_scalar_step(bc, SC_RESTART2, nb, tol2, delta2));
        return 0;
    };
    if (merged) CLV_CHECK(restart_merged());
    else {
        CLV_CUDA(cudaMemcpyAsync(p, r, nbytes, cudaMemcpyDeviceToDevice, st));
        CLV_CUDA(cudaMemcpyAsync(r0, r, nbytes, cudaMemcpyDeviceToDevice, st));
    }
    CLV_CUDA(cudaEventRecord(W->ev[2], st));
    CLV_CHECK(fetch_scalars(W, B, st));

    auto all_done = [&]() { for (int i = 0; i < B; i++) if (!W->sc_host[i].done) return false; return true; };
    // reliable update when any active rhs asks for one (delta rule), or when every active rhs claims convergence; a claim
    // that has waited 3 iterations for the others is confirmed anyway
    int claim_age = 0;
    bool last_any_claim = false, last_all_claim = false;
    auto any_update = [&]() {
        bool any_want = false, any_claim = false, all_claim = true;
        for (int i = 0; i < B; i++) {
            const RhsScalars &q = W->sc_host[i];
            if (q.done) continue;
            any_want |= q.want_update != 0;
            any_claim |= q.claim != 0;
            all_claim &= q.claim != 0;
        }
        claim_age = any_claim ? claim_age + 1 : 0;
        last_any_claim = any_claim;
        last_all_claim = all_claim;
        return any_want || all_claim || claim_age >= 3;
    };
    double ms_reliable = 0, ms_confirm = 0;
    bool verified = false;
    // odd sites and verification on the full lattice, all fp64: psi_o = A_oo^-1 (eta_o + kappa H_oe y), then ||eta - D psi||^2 out of
    // the epilogues of the two Dslash launches that apply D (residual variant without a store), their per-block partials reduced
    // together by the scalar step (SC_FINAL: report; SC_CONFIRM: also decide convergence)
    auto verify = [&](int step) -> int {
        CLV_CHECK(launch_dslash<double>(ctx, dargs<double>(y, eta_o, psi_o, ctx->kappa, 1, XM_PLAIN, 1), B, st, nullptr));
        CLV_CHECK(launch_dslash<double>(ctx, dargs<double>(psi_o, y, nullptr, -ctx->kappa, 0, XM_CLOVER, 0, DOT_RES, eta_e, W->partial), B, st, &grid));
        if (2 * grid > W->partial_blocks) {
            set_error("solve: partial buffer too small for the verification (%d blocks)", grid);
            return CLOVER_EINVAL;
        }
        CLV_CHECK(launch_dslash<double>(ctx, dargs<double>(y, psi_o, nullptr, -ctx->kappa, 1, XM_CLOVER, 0, DOT_RES, eta_o, W->partial + (size_t)grid * B * 4), B,
                                        st, nullptr));
        nl += 3;
        CLV_CHECK(blas_scalar_step(bc, step, 2 * grid, tol2, delta2));
        return 0;
    };
    // one BiCGStab iteration: [p update] Mhat p, alpha, s, Mhat s, omega, x/r update, rho/beta/flags, flag read-back
    auto iteration = [&](bool with_p, cudaEvent_t *kev) -> int {
        if (merged) {  // Mhat p (+ s), Mhat s (+ omega, rho', beta), x/r/p update (+ <q0,p>, ||r||^2), alpha/flags + their read-back
            CLV_CHECK(mhat<R>(ctx, B, p, tmp, v, DOT_S, r, nullptr, &grid, st, kev, nullptr, s, nullptr, W->sc_dev));
            CLV_CHECK(mhat<R>(ctx, B, s, tmp, t, DOT_XW, r0, W->partial, &grid, st, kev ? kev + 3 : nullptr, nullptr, nullptr, W->partial2));
            CLV_CHECK(blas_scalar_step(bc, SC_OMEGA2, grid, tol2, delta2));
            CLV_CHECK(blas_xrp_update<R>(bc, x, r, p, s, t, q0, &nb));
            CLV_CHECK(blas_scalar_step(bc, SC_RHO2, nb, tol2, delta2, W->sc_host_dev));   // + flag read-back (no publish launch)
            return 0;
        }
        if (with_p) CLV_CHECK(blas_p_update<R>(bc, p, r, v));
        CLV_CHECK(mhat<R>(ctx, B, p, tmp, v, DOT_W, r0, W->partial, &grid, st, kev));
        CLV_CHECK(blas_scalar_step(bc, SC_ALPHA, grid, tol2, delta2));
        CLV_CHECK(blas_s_update<R>(bc, r, v, s));
        CLV_CHECK(mhat<R>(ctx, B, s, tmp, t, DOT_X, nullptr, W->partial, &grid, st, kev ? kev + 3 : nullptr));
        CLV_CHECK(blas_scalar_step(bc, SC_OMEGA, grid, tol2, delta2));
        CLV_CHECK(blas_xr_update<R>(bc, x, r, p, s, t, r0, &nb));
        CLV_CHECK(blas_scalar_step(bc, SC_RHO, nb, tol2, delta2));
        CLV_CHECK(publish_scalars(W, B, st));
        return 0;
    };
    if (use_graph && (!W->iter_graph || W->graph_B != B || W->graph_prec != (int)sizeof(R) || W->graph_tol2 != tol2 || W->graph_delta2 != delta2 ||
                      W->graph_merged != (int)merged)) {
        if (W->iter_graph) { cudaGraphExecDestroy(W->iter_graph); W->iter_graph = nullptr; }
        const long long nl0 = nl;
        cudaGraph_t graph = nullptr;
        CLV_CUDA(cudaStreamBeginCapture(st, cudaStreamCaptureModeRelaxed));
        const int rc = iteration(true, nullptr);
        const cudaError_t ce = cudaStreamEndCapture(st, &graph);
        if (rc < 0) { if (graph) cudaGraphDestroy(graph); return rc; }
        CLV_CUDA(ce);
        W->graph_kernels = (int)(nl - nl0);
        nl = nl0;  // capturing launched nothing
        const cudaError_t ie = cudaGraphInstantiate(&W->iter_graph, graph, 0);
        cudaGraphDestroy(graph);
        CLV_CUDA(ie);
        W->graph_B = B; W->graph_prec = (int)sizeof(R); W->graph_tol2 = tol2; W->graph_delta2 = delta2; W->graph_merged = (int)merged;
    }
    bool need_p = merged;  // textbook ordering: p = r before the first iteration (no p update); merged: every iteration is alike
    // Merged iteration on lattices that are not launch-bound: its first Dslash (tmp = A^-1 H p) depends on nothing the host decides
    // after an iteration except a restart (a reliable update changes x, y and r, never p or tmp), so the one of iteration i+1 is
    // queued BEFORE the host waits for the flags of iteration i and the device does not idle during the round trip.  Not done while
    // a rhs claims convergence (the batch is about to end; a speculative launch after the last iteration is merely wasted).
    bool k1_queued = false;
    auto dslash_k1 = [&](int e) -> int {
        CLV_CUDA(cudaEventRecord(W->kev1[e][0], st));
        CLV_CHECK(launch_dslash<R>(ctx, dargs<R>(p, nullptr, tmp, (R)1, 1, XM_NONE, 1), B, st, nullptr));
        CLV_CUDA(cudaEventRecord(W->kev1[e][1], st));
        nl++;
        return 0;
    };
    auto iteration_after_k1 = [&]() -> int {
        const R k2 = (R)(-ctx->kappa * ctx->kappa);
        DslashArgs<R> a2 = dargs<R>(tmp, p, v, k2, 0, XM_CLOVER, 0, DOT_S, r, nullptr);
        a2.out2 = s;
        a2.sc = W->sc_dev;
        CLV_CUDA(cudaEventRecord(W->kev[1], st));
        CLV_CHECK(launch_dslash<R>(ctx, a2, B, st, nullptr));
        CLV_CUDA(cudaEventRecord(W->kev[2], st));
        CLV_CHECK(launch_dslash<R>(ctx, dargs<R>(s, nullptr, tmp, (R)1, 1, XM_NONE, 1), B, st, nullptr));
        CLV_CUDA(cudaEventRecord(W->kev[4], st));
        DslashArgs<R> a4 = dargs<R>(tmp, s, t, k2, 0, XM_CLOVER, 0, DOT_XW, r0, W->partial);
        a4.partial2 = W->partial2;
        CLV_CHECK(launch_dslash<R>(ctx, a4, B, st, &grid));
        CLV_CUDA(cudaEventRecord(W->kev[5], st));
        nl += 3;
        CLV_CHECK(blas_scalar_step(bc, SC_OMEGA2, grid, tol2, delta2));
        CLV_CUDA(cudaEventRecord(W->kev[0], st));
        CLV_CHECK(blas_xrp_update<R>(bc, x, r, p, s, t, q0, &nb));
        CLV_CUDA(cudaEventRecord(W->kev[3], st));
        CLV_CHECK(blas_scalar_step(bc, SC_RHO2, nb, tol2, delta2, W->sc_host_dev));
        CLV_CUDA(cudaEventRecord(W->ev_flags, st));
        return 0;
    };
    while (!all_done() && iters < max_iter) {
        if (merged && !use_graph) {
            const int e = iters & 1;
            if (!k1_queued) CLV_CHECK(dslash_k1(e));
            CLV_CHECK(iteration_after_k1());
            k1_queued = !last_any_claim && iters + 1 < max_iter;
            if (k1_queued) CLV_CHECK(dslash_k1(e ^ 1));
            CLV_CUDA(cudaEventSynchronize(W->ev_flags));
            clover_solve_stats &S = ctx->stats;
            CLV_CUDA(cudaEventElapsedTime(&ms, W->kev1[e][0], W->kev1[e][1])); S.ms_ainv_hop += ms;
            CLV_CUDA(cudaEventElapsedTime(&ms, W->kev[2], W->kev[4])); S.ms_ainv_hop += ms;
            CLV_CUDA(cudaEventElapsedTime(&ms, W->kev[1], W->kev[2])); S.ms_a_minus_hop_s += ms;
            CLV_CUDA(cudaEventElapsedTime(&ms, W->kev[4], W->kev[5])); S.ms_a_minus_hop += ms;
            CLV_CUDA(cudaEventElapsedTime(&ms, W->kev[0], W->kev[3])); S.ms_xrp_update += ms;
            S.n_ainv_hop += 2; S.n_a_minus_hop_s++; S.n_a_minus_hop++; S.n_xrp_update++;
        } else if (use_graph && need_p) {
            CLV_CUDA(cudaGraphLaunch(W->iter_graph, st));
            nl += W->graph_kernels;
            CLV_CUDA(cudaStreamSynchronize(st));
        } else {
            CLV_CHECK(iteration(need_p, use_graph ? nullptr : W->kev));
            CLV_CUDA(cudaStreamSynchronize(st));
            if (!use_graph) {
                for (int h = 0; h < 2; h++) {
                    CLV_CUDA(cudaEventElapsedTime(&ms, W->kev[3 * h], W->kev[3 * h + 1])); ctx->stats.ms_ainv_hop += ms;
                    CLV_CUDA(cudaEventElapsedTime(&ms, W->kev[3 * h + 1], W->kev[3 * h + 2]));
                    if (merged && h == 0) { ctx->stats.ms_a_minus_hop_s += ms; ctx->stats.n_a_minus_hop_s++; }
                    else { ctx->stats.ms_a_minus_hop += ms; ctx->stats.n_a_minus_hop++; }
                }
                ctx->stats.n_ainv_hop += 2;
            }
        }
        iters++;
        need_p = true;
        if (any_update() || iters == max_iter) {
            // reliable update: y += x, x = 0, r = b - Mhat y in fp64 (S 8(c) O6')
            CLV_CUDA(cudaEventRecord(W->ev[4], st));
            CLV_CHECK(blas_accumulate_y<R>(bc, y, x));
            if (last_all_claim && iters < max_iter) {
                // every active rhs claims convergence: confirm it with what the solve ends with anyway -- the odd sites and the fp64
                // residual on the full lattice (with exact odd sites it IS the even-odd residual (b - Mhat y, 0), R10) -- instead of
                // an even-odd recomputation followed by the same verification.  A rhs that fails goes on with a reliable update.
                CLV_CHECK(verify(SC_CONFIRM));
                CLV_CUDA(cudaEventRecord(W->ev[5], st));
                CLV_CHECK(fetch_scalars(W, B, st));
                CLV_CUDA(cudaEventElapsedTime(&ms, W->ev[4], W->ev[5]));
                ms_confirm += ms;
                if (all_done()) { verified = true; updates++; break; }
                CLV_CUDA(cudaEventRecord(W->ev[4], st));
            }
            // r = b - Mhat y with ||r||^2, fused into the epilogue of the second fp64 Dslash and stored in the iteration precision
            CLV_CHECK(mhat<double>(ctx, B, y, tmp64, sizeof(R) == 8 ? (double2 *)r : nullptr, DOT_RES, b, W->partial, &grid, st, nullptr,
                                   sizeof(R) == 4 ? (float4 *)r : nullptr));
            CLV_CHECK(blas_scalar_step(bc, SC_TRUE, grid, tol2, delta2));
            CLV_CUDA(cudaEventRecord(W->ev[5], st));
            CLV_CHECK(fetch_scalars(W, B, st));
            CLV_CUDA(cudaEventElapsedTime(&ms, W->ev[4], W->ev[5]));
            ms_reliable += ms;
            updates++;
            claim_age = 0;
        }
        {   // breakdown recovery (R11): r0 := r, rho := ||r||^2 for the rhs that asked for it; beta is already 0 so p := r next
            bool any_restart = false;
            for (int i = 0; i < B; i++) any_restart |= !W->sc_host[i].done && W->sc_host[i].restart == 1;
            if (any_restart) {
                if (merged) { CLV_CHECK(restart_merged()); k1_queued = false; }   // p changed, tmp was scratch
                else {
                    CLV_CHECK(blas_restart<R>(bc, r, r0));
                    CLV_CHECK(blas_scalar_step(bc, SC_RESTART, 0, tol2, delta2));
                }
            }
        }
    }
    CLV_CUDA(cudaEventRecord(W->ev[3], st));
    if (!verified) CLV_CHECK(verify(SC_FINAL));
    CLV_CUDA(cudaEventRecord(W->ev[4], st));
    CLV_CHECK((reorder_out<double, double>(g, dst, y, psi_o, B, st)));
    nl++;
    CLV_CUDA(cudaEventRecord(W->ev[5], st));
    CLV_CHECK(fetch_scalars(W, B, st));

    clover_solve_stats &S = ctx->stats;
    CLV_CUDA(cudaEventElapsedTime(&ms, W->ev[0], W->ev[1])); S.ms_reorder += ms;
    CLV_CUDA(cudaEventElapsedTime(&ms, W->ev[4], W->ev[5])); S.ms_reorder += ms;
    CLV_CUDA(cudaEventElapsedTime(&ms, W->ev[1], W->ev[2])); S.ms_prep += ms;
    CLV_CUDA(cudaEventElapsedTime(&ms, W->ev[2], W->ev[3])); S.ms_iterate += ms - ms_reliable - ms_confirm;
    S.ms_reliable += ms_reliable;
    CLV_CUDA(cudaEventElapsedTime(&ms, W->ev[3], W->ev[4])); S.ms_finish += ms + ms_confirm;
    CLV_CUDA(cudaEventElapsedTime(&ms, W->ev[0], W->ev[5])); S.ms_total += ms;

    int bad = 0;
    for (int i = 0; i < B; i++) {
        const RhsScalars &q = W->sc_host[i];
        clover_rhs_info &o = info[i];
        o.iters = iters;
        o.reliable_updates = updates;
        o.iter_resid = q.eta2 > 0 ? sqrt(q.true_r2 / q.eta2) : 0.0;
        o.true_resid = q.eta2 > 0 ? sqrt(q.r2 / q.eta2) : 0.0;
        o.status = q.status;
        if (o.status == 0 && !(o.true_resid <= tol)) o.status = (o.true_resid == o.true_resid) ? 1 : 3;
        if (o.status != 0) bad++;
    }
    return bad;
}

// greedy split of n into batches from {8,4,2,1} not exceeding `batch`
static int next_batch(int remaining, int batch)
{
    int b = 1;
    while (b * 2 <= batch && b * 2 <= remaining) b *= 2;
    return b;
}

int solve_batches(clover_ctx *ctx, const double *src, double *dst, int n_rhs, double tol, int max_iter, int batch, int mixed, clover_rhs_info *info,
                  cudaStream_t st, int host_buffers)
{
    CLV_CHECK(ensure_work(ctx, batch, mixed ? 4 : 8, host_buffers != 0, st));
    SolveWork *W = ctx->work;
    memset(&ctx->stats, 0, sizeof ctx->stats);
    const size_t per_rhs = (size_t)2 * ctx->geom.Vh * 24;  // doubles per canonical spinor
    int bad = 0, lastB = -1;
    if (!host_buffers) {
        for (int done = 0; done < n_rhs;) {
            const int B = next_batch(n_rhs - done, batch);
            if (B != lastB) CLV_CHECK(clear_fields(W, ctx->geom, B, st));
            lastB = B;
            int rc = mixed ? solve_batch<float>(ctx, src + done * per_rhs, dst + done * per_rhs, B, tol, max_iter, info + done, st)
                           : solve_batch<double>(ctx, src + done * per_rhs, dst + done * per_rhs, B, tol, max_iter, info + done, st);
            if (rc < 0) return rc;
            bad += rc;
            done += B;
        }
        return bad;
    }
    // host buffers: software pipeline over batches.  solve_batch synchronises `st` before it returns, so when batch i
    // starts, batch i-1 no longer reads stage_in[(i+1)&1] and its result sits complete in stage_out[(i-1)&1].
    CLV_CUDA(cudaStreamSynchronize(st));  // everything the caller queued on `st` before this call has happened
    int nb = 0, start[64], size[64];
    for (int done = 0; done < n_rhs && nb < 64; done += size[nb - 1]) { start[nb] = done; size[nb] = next_batch(n_rhs - done, batch); nb++; }
    if (nb == 64 && start[63] + size[63] < n_rhs) { set_error("clover_solve_host: more than 64 batches in one call"); return CLOVER_EINVAL; }
    auto h2d = [&](int i) -> cudaError_t {
        const cudaError_t e = cudaMemcpyAsync(W->stage_in[i & 1], src + start[i] * per_rhs, per_rhs * size[i] * sizeof(double), cudaMemcpyHostToDevice, W->s_in);
        return e != cudaSuccess ? e : cudaEventRecord(W->ev_in[i & 1], W->s_in);
    };
    // an error return must not leave copies in flight that read or write the caller's host buffers
    auto drain = [&]() { cudaStreamSynchronize(W->s_in); cudaStreamSynchronize(W->s_out); };
#define CLV_CUDA_DRAIN(call)                                                                                    \
    do {                                                                                                        \
        const cudaError_t e_ = (call);                                                                          \
        if (e_ != cudaSuccess) {                                                                                \
            drain();                                                                                            \
            set_error("%s failed at %s:%d: %s", #call, __FILE__, __LINE__, cudaGetErrorString(e_));             \
            return (e_ == cudaErrorMemoryAllocation) ? CLOVER_ENOMEM : CLOVER_ECUDA;                            \
        }                                                                                                       \
    } while (0)
    CLV_CUDA_DRAIN(h2d(0));
    for (int i = 0; i < nb; i++) {
        const int B = size[i], k = i & 1;
        if (i + 1 < nb) CLV_CUDA_DRAIN(h2d(i + 1));
        if (B != lastB) { const int rc = clear_fields(W, ctx->geom, B, st); if (rc < 0) { drain(); return rc; } }
        lastB = B;
        CLV_CUDA_DRAIN(cudaStreamWaitEvent(st, W->ev_in[k], 0));
        if (i >= 2) CLV_CUDA_DRAIN(cudaStreamWaitEvent(st, W->ev_out[k], 0));  // D2H of batch i-2 has drained stage_out[k]
        int rc = mixed ? solve_batch<float>(ctx, W->stage_in[k], W->stage_out[k], B, tol, max_iter, info + start[i], st)
                       : solve_batch<double>(ctx, W->stage_in[k], W->stage_out[k], B, tol, max_iter, info + start[i], st);
        if (rc < 0) { drain(); return rc; }
        bad += rc;
        CLV_CUDA_DRAIN(cudaMemcpyAsync(dst + start[i] * per_rhs, W->stage_out[k], per_rhs * B * sizeof(double), cudaMemcpyDeviceToHost, W->s_out));
        CLV_CUDA_DRAIN(cudaEventRecord(W->ev_out[k], W->s_out));
    }
#undef CLV_CUDA_DRAIN
    CLV_CUDA(cudaStreamSynchronize(W->s_out));
    return bad;
}

// ---- dslash_apply: canonical in -> op -> canonical out --------------------------------------------------------
template <typename R> struct Canon;
template <> struct Canon<float> { typedef float T; };
template <> struct Canon<double> { typedef double T; };

template <typename R> static int apply_chunk(clover_ctx *ctx, int op, const R *in, R *out, int B, cudaStream_t st)
{
    typedef typename Vec<R>::T V;
    SolveWork *W = ctx->work;
    const Geom &g = ctx->geom;
    V *ie, *io, *oe, *oo, *tmp;
    if (sizeof(R) == 8) {
        ie = (V *)W->f64[0]; io = (V *)W->f64[1]; oe = (V *)W->f64[2]; oo = (V *)W->f64[3]; tmp = (V *)W->f64[4];
    } else {
        ie = (V *)W->sl[0]; io = (V *)W->sl[1]; oe = (V *)W->sl[2]; oo = (V *)W->sl[3]; tmp = (V *)W->sl[4];
    }
    CLV_CHECK((reorder_in<R, R>(g, in, ie, io, B, st)));
    const R one = (R)1, mk_ = (R)(-ctx->kappa), mk2 = (R)(-ctx->kappa * ctx->kappa);
    const V *re = nullptr, *ro = nullptr;
    switch (op) {
    case CLOVER_OP_HOP_EO:
        CLV_CHECK(launch_dslash<R>(ctx, dargs<R>(io, nullptr, oe, one, 0, XM_NONE, 0), B, st, nullptr));
        re = oe;
        break;
    case CLOVER_OP_HOP_OE:
        CLV_CHECK(launch_dslash<R>(ctx, dargs<R>(ie, nullptr, oo, one, 1, XM_NONE, 0), B, st, nullptr));
        ro = oo;
        break;
    case CLOVER_OP_HOP_FULL:
        CLV_CHECK(launch_dslash<R>(ctx, dargs<R>(io, nullptr, oe, one, 0, XM_NONE, 0), B, st, nullptr));
        CLV_CHECK(launch_dslash<R>(ctx, dargs<R>(ie, nullptr, oo, one, 1, XM_NONE, 0), B, st, nullptr));
        re = oe; ro = oo;
        break;
    case CLOVER_OP_CLOVER:
    case CLOVER_OP_CLOVER_INV:
        CLV_CHECK(launch_clover<R>(ctx, ie, oe, 0, op == CLOVER_OP_CLOVER_INV, B, st));
        CLV_CHECK(launch_clover<R>(ctx, io, oo, 1, op == CLOVER_OP_CLOVER_INV, B, st));
        re = oe; ro = oo;
        break;
    case CLOVER_OP_D_FULL:
        CLV_CHECK(launch_dslash<R>(ctx, dargs<R>(io, ie, oe, mk_, 0, XM_CLOVER, 0), B, st, nullptr));
        CLV_CHECK(launch_dslash<R>(ctx, dargs<R>(ie, io, oo, mk_, 1, XM_CLOVER, 0), B, st, nullptr));
        re = oe; ro = oo;
        break;
    case CLOVER_OP_MHAT:
        CLV_CHECK(launch_dslash<R>(ctx, dargs<R>(ie, nullptr, tmp, one, 1, XM_NONE, 1), B, st, nullptr));
        CLV_CHECK(launch_dslash<R>(ctx, dargs<R>(tmp, ie, oe, mk2, 0, XM_CLOVER, 0), B, st, nullptr));
        re = oe;
        break;
    default:
        set_error("dslash_apply: unknown op %d", op);
        return CLOVER_EINVAL;
    }
    CLV_CHECK((reorder_out<R, R>(g, out, re, ro, B, st)));
    return 0;
}

int apply_op(clover_ctx *ctx, int op, int precision, const void *in, void *out, int n_rhs, cudaStream_t st)
{
    CLV_CHECK(ensure_work(ctx, std::min(8, ctx->max_rhs), 4, false, st));
    const size_t per_rhs = (size_t)2 * ctx->geom.Vh * 24;
    int lastB = -1;
    for (int done = 0; done < n_rhs;) {
        const int B = next_batch(n_rhs - done, ctx->max_rhs);
        if (B != lastB) CLV_CHECK(clear_fields(ctx->work, ctx->geom, B, st));
        lastB = B;
        if (precision == 32) CLV_CHECK(apply_chunk<float>(ctx, op, (const float *)in + done * per_rhs, (float *)out + done * per_rhs, B, st));
        else CLV_CHECK(apply_chunk<double>(ctx, op, (const double *)in + done * per_rhs, (double *)out + done * per_rhs, B, st));
        done += B;
    }
    return 0;
}

// ---- kernel benchmark on internal-layout scratch fields ----------------------------------------------------------
template <typename R> __global__ void fill_kernel(R *f, size_t n, unsigned salt)
{
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        unsigned h = (unsigned)i * 2654435761u + salt;
        h ^= h >> 15; h *= 2246822519u; h ^= h >> 13;
        f[i] = (R)((int)(h & 0xffff) - 32768) * (R)(1.0 / 32768.0);
    }
}

template <typename R> static int bench_impl(clover_ctx *ctx, int kernel, int B, int reps, int flush_l2, float *ms_out, cudaStream_t st)
{
    typedef typename Vec<R>::T V;
    SolveWork *W = ctx->work;
    const Geom &g = ctx->geom;
    V *f[4];
    for (int i = 0; i < 4; i++) f[i] = sizeof(R) == 8 ? (V *)W->f64[i] : (V *)W->sl[i];
    CLV_CHECK(clear_fields(W, g, B, st));
    const size_t nreal = (size_t)((unsigned)g.Vh * B / 32u) * 32u * 24u;  // whole lane blocks only: padding lanes stay zero
    for (int i = 0; i < 3; i++) fill_kernel<R><<<1184, 256, 0, st>>>((R *)f[i], nreal, 17u * i + 1u);
    CLV_CUDA(cudaGetLastError());
    const size_t flush_bytes = (size_t)256 << 20;
    if (flush_l2 && !W->flush) CLV_CUDA(cudaMalloc(&W->flush, flush_bytes));
    DslashArgs<R> a;
    const R k2 = (R)(-ctx->kappa * ctx->kappa);
    switch (kernel) {
    case CLOVER_KERNEL_HOP: a = dargs<R>(f[0], nullptr, f[3], (R)1, 0, XM_NONE, 0); break;
    case CLOVER_KERNEL_AINV_HOP: a = dargs<R>(f[0], nullptr, f[3], (R)1, 1, XM_NONE, 1); break;
    case CLOVER_KERNEL_A_MINUS_HOP: a = dargs<R>(f[0], f[1], f[3], k2, 0, XM_CLOVER, 0, DOT_X, nullptr, W->partial); break;
    case CLOVER_KERNEL_A_MINUS_HOP_S:
        a = dargs<R>(f[0], f[1], f[3], k2, 0, XM_CLOVER, 0, DOT_S, f[2]);
        a.out2 = f[3];
        a.sc = W->sc_dev;
        break;
    case CLOVER_KERNEL_A_MINUS_HOP_XW:
        a = dargs<R>(f[0], f[1], f[3], k2, 0, XM_CLOVER, 0, DOT_XW, f[2], W->partial);
        a.partial2 = W->partial2;
        break;
    default: set_error("clover_bench_kernel: unknown kernel %d", kernel); return CLOVER_EINVAL;
    }
    double total = 0;
    for (int it = -3; it < reps; it++) {  // 3 warm-up launches
        if (flush_l2) CLV_CUDA(cudaMemsetAsync(W->flush, it & 0xff, flush_bytes, st));
        CLV_CUDA(cudaEventRecord(W->ev[0], st));
        CLV_CHECK(launch_dslash<R>(ctx, a, B, st, nullptr));
        CLV_CUDA(cudaEventRecord(W->ev[1], st));
        CLV_CUDA(cudaEventSynchronize(W->ev[1]));
        float ms;
        CLV_CUDA(cudaEventElapsedTime(&ms, W->ev[0], W->ev[1]));
        if (it >= 0) total += ms;
    }
    *ms_out = (float)(total / reps);
    return 0;
}

int bench_kernel(clover_ctx *ctx, int kernel, int precision, int n_rhs, int reps, int flush_l2, float *ms, cudaStream_t st)
{
    CLV_CHECK(ensure_work(ctx, n_rhs, 4, false, st));
    return precision == 32 ? bench_impl<float>(ctx, kernel, n_rhs, reps, flush_l2, ms, st) : bench_impl<double>(ctx, kernel, n_rhs, reps, flush_l2, ms, st);
}

}  // namespace clv
