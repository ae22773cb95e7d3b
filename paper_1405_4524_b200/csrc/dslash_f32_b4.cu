// generated instantiation unit: Dslash kernels for float, 4 right-hand sides per site
#include "dslash_inst.cuh"
namespace clv {
template int launch_dslash_B<float, 4>(const clover_ctx *, const DslashArgs<float> &, cudaStream_t, int *);
template int launch_clover_B<float, 4>(const clover_ctx *, const Vec<float>::T *, Vec<float>::T *, int, int, cudaStream_t);
}  // namespace clv
