// generated instantiation unit: Dslash kernels for double, 2 right-hand sides per site
#include "dslash_inst.cuh"
namespace clv {
template int launch_dslash_B<double, 2>(const clover_ctx *, const DslashArgs<double> &, cudaStream_t, int *);
template int launch_clover_B<double, 2>(const clover_ctx *, const Vec<double>::T *, Vec<double>::T *, int, int, cudaStream_t);
}  // namespace clv
