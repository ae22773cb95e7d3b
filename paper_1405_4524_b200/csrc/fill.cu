// fill.cu -- the outer-product "fill" of the stochastic all-to-all propagator, arXiv:1405.4524 eq. 7.3 ("S_s fill"
// and "S_s^dagger fill" of Tables I-II):
//     S(t,z,a; t0,x,b) = (1/(N_r scale^2)) sum_i X_i(t,z,a) conj(eta_i(t0,x,b))
// i.e. C[m][n] = norm * sum_k A[k][m] conj(B[k][n]) with A[k] = X_k (the whole canonical spinor, M = 12 V contiguous),
// B[k] = eta_k restricted to timeslice t0 (N = 12 L^3 contiguous), K = N_r: a complex rank-N_r update whose 16-byte outputs are
// written once.  The dagger version C'[n][m] = conj(C[m][n]) = norm * sum_k B[k][n] conj(A[k][m]) is the same kernel with the
// operands swapped, so its stores are coalesced as well.  fp64 throughout (the propagators are fp64; parity 1e-13).
// The paper accumulates one source at a time (a rank-1 update of the 9.7 GB array per source at L = 8: 100.8 s CPU, 8.8 s GPU,
// Table II); here all N_r sources go through one pass, so the array is written once.
#include "context.h"

namespace clv {

constexpr int FL_TILE = 64;     // outputs per CTA: 64 x 64
constexpr int FL_KT = 8;        // sources staged per step
constexpr int FL_THREADS = 256; // 16 x 16 threads, 4 x 4 outputs each at {ti + 16 a} x {tj + 16 b}

// C[m*ldc + n] = norm * sum_k A[k*lda + m] * conj(B[k*ldb + n]),  m < M, n < N
__global__ void __launch_bounds__(FL_THREADS, 2) fill_gemm_kernel(const double2 *__restrict__ A, long lda, const double2 *__restrict__ B, long ldb, int K,
                                                                long M, long N, double norm, double2 *__restrict__ C, long ldc)
{
    __shared__ __align__(16) double2 As[FL_KT][FL_TILE], Bs[FL_KT][FL_TILE];
    const long m0 = (long)blockIdx.y * FL_TILE, n0 = (long)blockIdx.x * FL_TILE;
    const int ti = threadIdx.x >> 4, tj = threadIdx.x & 15;
    double2 acc[4][4];
#pragma unroll
    for (int a = 0; a < 4; a++)
#pragma unroll
        for (int b = 0; b < 4; b++) acc[a][b] = make_double2(0., 0.);
    for (int kb = 0; kb < K; kb += FL_KT) {
        // 8 x 64 elements per operand, 2 + 2 per thread; a warp reads 512 contiguous bytes of one source
#pragma unroll
        for (int it = 0; it < 2; it++) {
            const int item = threadIdx.x + FL_THREADS * it, kk = item >> 6, col = item & 63;
            double2 a = make_double2(0., 0.), b = make_double2(0., 0.);
            if (kb + kk < K) {
                if (m0 + col < M) a = __ldg(A + (long)(kb + kk) * lda + m0 + col);
                if (n0 + col < N) b = __ldg(B + (long)(kb + kk) * ldb + n0 + col);
            }
            As[kk][col] = a;
            Bs[kk][col] = make_double2(b.x, -b.y);   // conj
        }
        __syncthreads();
#pragma unroll
        for (int kk = 0; kk < FL_KT; kk++) {
            double2 a[4], b[4];
#pragma unroll
            for (int r = 0; r < 4; r++) {
                a[r] = As[kk][ti + 16 * r];
                b[r] = Bs[kk][tj + 16 * r];
            }
#pragma unroll
            for (int x = 0; x < 4; x++)
#pragma unroll
                for (int y = 0; y < 4; y++) {
                    acc[x][y].x += a[x].x * b[y].x;
                    acc[x][y].x -= a[x].y * b[y].y;
                    acc[x][y].y += a[x].x * b[y].y;
                    acc[x][y].y += a[x].y * b[y].x;
                }
        }
        __syncthreads();
    }
#pragma unroll
    for (int x = 0; x < 4; x++) {
        const long m = m0 + ti + 16 * x;
        if (m >= M) continue;
#pragma unroll
        for (int y = 0; y < 4; y++) {
            const long n = n0 + tj + 16 * y;
            if (n < N) C[m * ldc + n] = make_double2(norm * acc[x][y].x, norm * acc[x][y].y);   // 16 lanes -> 256 contiguous bytes
        }
    }
}

int launch_fill(const double *x, const double *eta, const int dims[4], int n, int t0, double scale, int dagger, double *s, cudaStream_t st)
{
    const long V3 = (long)dims[0] * dims[1] * dims[2], V = V3 * dims[3];
    const long M = 12 * V, N = 12 * V3;              // rows (t, z, a), columns (x, b)
    const double2 *A = (const double2 *)x, *B = (const double2 *)eta + (long)t0 * N;
    const double norm = 1.0 / ((double)n * scale * scale);
    if (!dagger) {
        dim3 grid((unsigned)((N + FL_TILE - 1) / FL_TILE), (unsigned)((M + FL_TILE - 1) / FL_TILE));
        fill_gemm_kernel<<<grid, FL_THREADS, 0, st>>>(A, M, B, M, n, M, N, norm, (double2 *)s, N);
    } else {  // S^dagger[x, b, t, z, a]: rows (x, b), columns (t, z, a); operands swapped
        dim3 grid((unsigned)((M + FL_TILE - 1) / FL_TILE), (unsigned)((N + FL_TILE - 1) / FL_TILE));
        fill_gemm_kernel<<<grid, FL_THREADS, 0, st>>>(B, M, A, M, n, N, M, norm, (double2 *)s, M);
    }
    CLV_CUDA(cudaGetLastError());
    return 0;
}

}  // namespace clv
