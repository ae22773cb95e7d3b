// traces.cu -- the two trace operations of Table I of arXiv:1405.4524:
//   sum_y Tr[S_p(t,y;0,0) S_p^+(t,y;0,0)]   and   sum_x sum_z Tr[S_s(t,z;0,x) S_s^+(t,z;0,x)],
// "the dagger is only w.r.t. the spin-color indices" (L293): both are the squared Frobenius norm of everything on timeslice t,
//   out[t] = sum_{o < n_outer} sum_{k < slice_len} |f[o][t][k]|^2      for a complex128 field viewed as [n_outer][T][slice_len].
// A pure read stream (HBM bound): grid-stride 16-byte loads, fp64 accumulation, warp shuffle -> shared memory -> per-block
// partials -> fixed-order second stage (deterministic).
#include "context.h"
#include <algorithm>

namespace clv {

constexpr int TR_THREADS = 256;

__global__ void __launch_bounds__(TR_THREADS) timeslice_norm2_kernel(const double2 *__restrict__ f, long n_outer, int T, long slice_len,
                                                                    double *__restrict__ partial)
{
    __shared__ double sm[TR_THREADS / 32];
    const int t = blockIdx.y;
    double acc = 0;
    for (long o = 0; o < n_outer; o++) {
        const double2 *p = f + (o * T + t) * slice_len;
        for (long k = (long)blockIdx.x * TR_THREADS + threadIdx.x; k < slice_len; k += (long)gridDim.x * TR_THREADS) {
            const double2 v = __ldg(p + k);
            acc += v.x * v.x + v.y * v.y;
        }
    }
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, off);
    if ((threadIdx.x & 31) == 0) sm[threadIdx.x >> 5] = acc;
    __syncthreads();
    if (threadIdx.x == 0) {
        double s = 0;
        for (int w = 0; w < TR_THREADS / 32; w++) s += sm[w];
        partial[(long)t * gridDim.x + blockIdx.x] = s;
    }
}

__global__ void timeslice_norm2_reduce_kernel(const double *__restrict__ partial, int nblocks, double *__restrict__ out)
{
    const int t = blockIdx.x;
    if (threadIdx.x != 0) return;
    double s = 0;
    for (int b = 0; b < nblocks; b++) s += partial[(long)t * nblocks + b];
    out[t] = s;
}

// out[t] = sum a conj(b): the trace between fills from two independent source sets, same structure, two read streams
__global__ void __launch_bounds__(TR_THREADS) timeslice_inner_kernel(const double2 *__restrict__ a, const double2 *__restrict__ b, long n_outer, int T,
                                                                    long slice_len, double2 *__restrict__ partial)
{
    __shared__ double2 sm[TR_THREADS / 32];
    const int t = blockIdx.y;
    double re = 0, im = 0;
    for (long o = 0; o < n_outer; o++) {
        const long base = (o * T + t) * slice_len;
        for (long k = (long)blockIdx.x * TR_THREADS + threadIdx.x; k < slice_len; k += (long)gridDim.x * TR_THREADS) {
            const double2 u = __ldg(a + base + k), v = __ldg(b + base + k);
            re += u.x * v.x + u.y * v.y;
            im += __dmul_rn(u.y, v.x) - __dmul_rn(u.x, v.y);   // separately rounded products: exactly 0 when a = b
        }
    }
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
        re += __shfl_xor_sync(0xffffffffu, re, off);
        im += __shfl_xor_sync(0xffffffffu, im, off);
    }
    if ((threadIdx.x & 31) == 0) sm[threadIdx.x >> 5] = make_double2(re, im);
    __syncthreads();
    if (threadIdx.x == 0) {
        double sr = 0, si = 0;
        for (int w = 0; w < TR_THREADS / 32; w++) {
            sr += sm[w].x;
            si += sm[w].y;
        }
        partial[(long)t * gridDim.x + blockIdx.x] = make_double2(sr, si);
    }
}

__global__ void timeslice_inner_reduce_kernel(const double2 *__restrict__ partial, int nblocks, double2 *__restrict__ out)
{
    const int t = blockIdx.x;
    if (threadIdx.x != 0) return;
    double sr = 0, si = 0;
    for (int b = 0; b < nblocks; b++) {
        sr += partial[(long)t * nblocks + b].x;
        si += partial[(long)t * nblocks + b].y;
    }
    out[t] = make_double2(sr, si);
}

static int trace_blocks(int T, long slice_len)
{
    return (int)std::max<long>(1, std::min<long>((slice_len + TR_THREADS * 8 - 1) / (TR_THREADS * 8), (148L * 16 + T - 1) / T));
}

int launch_timeslice_inner(const double *a, const double *b, long n_outer, int T, long slice_len, double *out, cudaStream_t st)
{
    const int nblocks = trace_blocks(T, slice_len);
    double2 *partial = nullptr;
    CLV_CUDA(cudaMallocAsync((void **)&partial, sizeof(double2) * (size_t)T * nblocks, st));
    timeslice_inner_kernel<<<dim3(nblocks, T), TR_THREADS, 0, st>>>((const double2 *)a, (const double2 *)b, n_outer, T, slice_len, partial);
    CLV_CUDA(cudaGetLastError());
    timeslice_inner_reduce_kernel<<<T, 32, 0, st>>>(partial, nblocks, (double2 *)out);
    CLV_CUDA(cudaGetLastError());
    CLV_CUDA(cudaFreeAsync(partial, st));
    return 0;
}

int launch_timeslice_norm2(const double *f, long n_outer, int T, long slice_len, double *out, cudaStream_t st)
{
    const int nblocks = trace_blocks(T, slice_len);
    double *partial = nullptr;
    CLV_CUDA(cudaMallocAsync((void **)&partial, sizeof(double) * (size_t)T * nblocks, st));
    timeslice_norm2_kernel<<<dim3(nblocks, T), TR_THREADS, 0, st>>>((const double2 *)f, n_outer, T, slice_len, partial);
    CLV_CUDA(cudaGetLastError());
    timeslice_norm2_reduce_kernel<<<T, 32, 0, st>>>(partial, nblocks, out);
    CLV_CUDA(cudaGetLastError());
    CLV_CUDA(cudaFreeAsync(partial, st));
    return 0;
}

}  // namespace clv
