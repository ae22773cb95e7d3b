// dslash.cu -- runtime dispatch over the batch size to the per-(precision, B) instantiation units.
#include "dslash_kernel.cuh"

namespace clv {

template <typename R, int B>
int launch_clover_B(const clover_ctx *ctx, const typename Vec<R>::T *in, typename Vec<R>::T *out, int parity, int inverse, cudaStream_t st);

#define CLV_DECL(RT, B)                                                                                             \
    extern template int launch_dslash_B<RT, B>(const clover_ctx *, const DslashArgs<RT> &, cudaStream_t, int *);    \
    extern template int launch_clover_B<RT, B>(const clover_ctx *, const Vec<RT>::T *, Vec<RT>::T *, int, int, cudaStream_t);
CLV_DECL(float, 1) CLV_DECL(float, 2) CLV_DECL(float, 4) CLV_DECL(float, 8)
CLV_DECL(double, 1) CLV_DECL(double, 2) CLV_DECL(double, 4) CLV_DECL(double, 8)
#undef CLV_DECL

template <typename R> int launch_dslash(const clover_ctx *ctx, const DslashArgs<R> &a, int B, cudaStream_t st, int *grid_out)
{
    switch (B) {
    case 1: return launch_dslash_B<R, 1>(ctx, a, st, grid_out);
    case 2: return launch_dslash_B<R, 2>(ctx, a, st, grid_out);
    case 4: return launch_dslash_B<R, 4>(ctx, a, st, grid_out);
    case 8: return launch_dslash_B<R, 8>(ctx, a, st, grid_out);
    }
    set_error("dslash: batch must be 1, 2, 4 or 8 (got %d)", B);
    return CLOVER_EINVAL;
}
template int launch_dslash<float>(const clover_ctx *, const DslashArgs<float> &, int, cudaStream_t, int *);
template int launch_dslash<double>(const clover_ctx *, const DslashArgs<double> &, int, cudaStream_t, int *);

template <typename R>
int launch_clover(const clover_ctx *ctx, const typename Vec<R>::T *in, typename Vec<R>::T *out, int parity, int inverse, int B, cudaStream_t st)
{
    switch (B) {
    case 1: return launch_clover_B<R, 1>(ctx, in, out, parity, inverse, st);
    case 2: return launch_clover_B<R, 2>(ctx, in, out, parity, inverse, st);
    case 4: return launch_clover_B<R, 4>(ctx, in, out, parity, inverse, st);
    case 8: return launch_clover_B<R, 8>(ctx, in, out, parity, inverse, st);
    }
    set_error("clover: batch must be 1, 2, 4 or 8 (got %d)", B);
    return CLOVER_EINVAL;
}
template int launch_clover<float>(const clover_ctx *, const float4 *, float4 *, int, int, int, cudaStream_t);
template int launch_clover<double>(const clover_ctx *, const double2 *, double2 *, int, int, int, cudaStream_t);

int dslash_block_size() { return DSLASH_BLOCK; }

}  // namespace clv
