// fill.cu -- the outer-product "fill" of the stochastic all-to-all propagator, arXiv:1405.4524 eq. 7.3 ("S_s fill"
// and "S_s^dagger fill" of Tables I-II):
//     S(t,z,a; t0,x,b) = (1/(N_r scale^2)) sum_i X_i(t,z,a) conj(eta_i(t0,x,b))
// i.e. C[m][n] = norm * sum_k A[k][m] conj(B[k][n]) with A[k] = X_k (the whole canonical spinor, M = 12 V contiguous),
// B[k] = eta_k restricted to timeslice t0 (N = 12 L^3 contiguous), K = N_r: a complex rank-N_r update whose 16-byte outputs are
// written once.  The dagger version C'[n][m] = conj(C[m][n]) = norm * sum_k B[k][n] conj(A[k][m]) is the same kernel with the
// operands swapped, so its stores are coalesced as well.  fp64 throughout (the propagators are fp64; parity 1e-13), on the fp64
// tensor pipe (mma.sync m8n8k4, SASS DMMA: tcgen05 has no fp64 type).
// The paper accumulates one source at a time (a rank-1 update of the 9.7 GB array per source at L = 8: 100.8 s CPU, 8.8 s GPU,
// Table II); here all N_r sources go through one pass, so the array is written once.
#include "context.h"
#include <cuda_pipeline.h>

namespace clv {

constexpr int FL_TILE = 64;     // outputs per CTA: 64 x 64 complex, one 32 x 32 quadrant per warp (computed as two 32 x 16 halves)
constexpr int FL_KT = 32;       // sources staged per step (all of them at the paper's N_r <= 32)
constexpr int FL_LD = FL_TILE + 2;   // row stride of the shared tiles in complex numbers (8 words mod 32: the four source rows x two columns of a quarter-warp's 16-byte fragment loads fall in disjoint banks)
constexpr int FL_THREADS = 128;

// D (8x8, fp64) += A (8x4, row) B (4x8, col) on the fp64 tensor pipe (SASS DMMA); fragments per thread T: a = A[T/4][T%4], b = B[T%4][T/4],
// c/d = C[T/4][2 (T%4) + {0,1}]
__device__ __forceinline__ void fill_dmma884(double (&c)[2], double a, double b)
{
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};" : "+d"(c[0]), "+d"(c[1]) : "d"(a), "d"(b));
}

// C[m*ldc + n] = norm * sum_k A[k*lda + m] * conj(B[k*ldb + n]),  m < M, n < N.
// Three REAL GEMMs over the sources per complex one (Gauss' three-multiplication form: a quarter fewer DMMA than four products).  With
// a = ar + i ai, b = br + i bi:   a conj(b) = (ar br + ai bi) + i (ai br - ar bi) = (k1 - k3) + i (k1 + k2),
//   k1 = (ar + ai) br,   k2 = ar (-bi - br),   k3 = ai (br - bi);   the three sums over k sit in three accumulator sets, combined at the end.
__global__ void __launch_bounds__(FL_THREADS, 3) fill_gemm_kernel(const double2 *__restrict__ A, long lda, const double2 *__restrict__ B, long ldb, int K,
                                                                long M, long N, double norm, double2 *__restrict__ C, long ldc)
{
    extern __shared__ __align__(16) double2 fl_smem[];
    double2(*As)[FL_LD] = reinterpret_cast<double2(*)[FL_LD]>(fl_smem);
    double2(*Bs)[FL_LD] = reinterpret_cast<double2(*)[FL_LD]>(fl_smem + FL_KT * FL_LD);
    const long m0 = (long)blockIdx.y * FL_TILE, n0 = (long)blockIdx.x * FL_TILE;
    const int w = threadIdx.x >> 5, lane = threadIdx.x & 31, fr = lane >> 2, fk = lane & 3;
    const int wm = 32 * (w >> 1), wn = 32 * (w & 1);   // this warp's quadrant
    const bool single = K <= FL_KT;                    // the paper's case: every source staged at once, the two halves share the staging
    for (int half = 0; half < 2; half++) {             // columns [wn + 16 half, wn + 16 half + 16) of the quadrant
        double acc1[4][2][2], acc2[4][2][2], acc3[4][2][2];
#pragma unroll
        for (int x = 0; x < 4; x++)
#pragma unroll
            for (int y = 0; y < 2; y++)
#pragma unroll
                for (int e = 0; e < 2; e++) acc1[x][y][e] = acc2[x][y][e] = acc3[x][y][e] = 0.0;
        for (int kb = 0; kb < K; kb += FL_KT) {
            if (!(single && half == 1)) {
                if (half == 1 || kb > 0) __syncthreads();   // the previous block has been read
                // 32 x 64 elements per operand, 16-byte async copies; a warp copies 512 contiguous bytes of one source
#pragma unroll 4
                for (int it = 0; it < FL_KT * FL_TILE / FL_THREADS; it++) {
                    const int item = threadIdx.x + FL_THREADS * it, kk = item >> 6, col = item & 63;
                    double2 *da = &As[kk][col], *db = &Bs[kk][col];
                    if (kb + kk < K && m0 + col < M) __pipeline_memcpy_async(da, A + (long)(kb + kk) * lda + m0 + col, 16);
                    else *da = make_double2(0., 0.);
                    if (kb + kk < K && n0 + col < N) __pipeline_memcpy_async(db, B + (long)(kb + kk) * ldb + n0 + col, 16);
                    else *db = make_double2(0., 0.);
                }
                __pipeline_commit();
                __pipeline_wait_prior(0);
                __syncthreads();
            }
#pragma unroll 2
            for (int s = 0; s < FL_KT / 4; s++) {   // four sources per DMMA step; this lane's source = 4 s + fk
                double ar[4], ai[4], apq[4], br[2], bm[2], bp[2];
#pragma unroll
                for (int r = 0; r < 4; r++) {
                    const double2 a = As[4 * s + fk][wm + 8 * r + fr];
                    ar[r] = a.x; ai[r] = a.y; apq[r] = a.x + a.y;
                }
#pragma unroll
                for (int r = 0; r < 2; r++) {
                    const double2 b = Bs[4 * s + fk][wn + 16 * half + 8 * r + fr];
                    br[r] = b.x; bm[r] = -b.y - b.x; bp[r] = b.x - b.y;
                }
#pragma unroll
                for (int x = 0; x < 4; x++)
#pragma unroll
                    for (int y = 0; y < 2; y++) {
                        fill_dmma884(acc1[x][y], apq[x], br[y]);
                        fill_dmma884(acc2[x][y], ar[x], bm[y]);
                        fill_dmma884(acc3[x][y], ai[x], bp[y]);
                    }
            }
        }
        // a thread holds two neighbouring outputs (n, n + 1) of a row: 32 contiguous bytes; the 4 lanes of a row write one 128-byte line
#pragma unroll
        for (int x = 0; x < 4; x++) {
            const long m = m0 + wm + 8 * x + fr;
            if (m >= M) continue;
#pragma unroll
            for (int y = 0; y < 2; y++) {
                const long n = n0 + wn + 16 * half + 8 * y + 2 * fk;
                if (n < N) C[m * ldc + n] = make_double2(norm * (acc1[x][y][0] - acc3[x][y][0]), norm * (acc1[x][y][0] + acc2[x][y][0]));
                if (n + 1 < N) C[m * ldc + n + 1] = make_double2(norm * (acc1[x][y][1] - acc3[x][y][1]), norm * (acc1[x][y][1] + acc2[x][y][1]));
            }
        }
    }
}

int launch_fill(const double *x, const double *eta, const int dims[4], int n, int t0, double scale, int dagger, double *s, cudaStream_t st)
{
    const long V3 = (long)dims[0] * dims[1] * dims[2], V = V3 * dims[3];
    const long M = 12 * V, N = 12 * V3;              // rows (t, z, a), columns (x, b)
    const double2 *A = (const double2 *)x, *B = (const double2 *)eta + (long)t0 * N;
    const double norm = 1.0 / ((double)n * scale * scale);
    constexpr size_t smem = sizeof(double2) * 2 * FL_KT * FL_LD;
    static const cudaError_t attr = cudaFuncSetAttribute(fill_gemm_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    CLV_CUDA(attr);
    if (!dagger) {
        dim3 grid((unsigned)((N + FL_TILE - 1) / FL_TILE), (unsigned)((M + FL_TILE - 1) / FL_TILE));
        fill_gemm_kernel<<<grid, FL_THREADS, smem, st>>>(A, M, B, M, n, M, N, norm, (double2 *)s, N);
    } else {  // S^dagger[x, b, t, z, a]: rows (x, b), columns (t, z, a); operands swapped
        dim3 grid((unsigned)((M + FL_TILE - 1) / FL_TILE), (unsigned)((N + FL_TILE - 1) / FL_TILE));
        fill_gemm_kernel<<<grid, FL_THREADS, smem, st>>>(B, M, A, M, n, N, M, norm, (double2 *)s, M);
    }
    CLV_CUDA(cudaGetLastError());
    return 0;
}

}  // namespace clv
