// generated instantiation unit: Dslash kernels for double, 8 right-hand sides per site
#define CLV_BUILD_DSLASH3D
#include "dslash_inst.cuh"
namespace clv {
template int launch_dslash_B<double, 8>(const clover_ctx *, const DslashArgs<double> &, cudaStream_t, int *);
template int launch_clover_B<double, 8>(const clover_ctx *, const Vec<double>::T *, Vec<double>::T *, int, int, cudaStream_t);
}  // namespace clv
