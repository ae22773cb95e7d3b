// contract.cu -- stochastic-operator contraction of arXiv:1405.4524, eqs. 7.5-7.7, SURVEY 8(f) rank 1:
//   O_ij(t)   = sum_y eta_i^*(t,y) gamma5 X_j(t,y)            one complex number per (t, i, j)
//   C(t0, t)  = (1/(N_r^2 scale^4)) sum_ij O_ij(t) O_ji(t0)
// Per timeslice this is a complex GEMM  O(t) = conj(E_t) diag(gamma5) X_t^T  with M = N = N_r and K = 12 L^3 (the one dense
// contraction of the paper's pipeline).  The propagators come out of clover_solve in fp64 and parity is asked at 1e-13, so
// the product runs on the fp64 FMA pipe: tcgen05 has no fp64 path, and at N_r = 32 the arithmetic intensity
// (8 N_r^2 K flop over 32 N_r K bytes = N_r/4 flop/byte) sits at the fp64 ridge of a B200, not above it.
// Canonical layouts: eta, X = [n][T][Z][Y][X][4][3] complex128; O = [T][n][n] complex128; C = [T][T] complex128.
#include "context.h"
#include <algorithm>
#include <cuda_pipeline.h>

namespace clv {

constexpr int CT_TILE = 32;    // (i, j) tile edge
constexpr int CT_KT = 16;      // k elements staged per step
constexpr int CT_THREADS = 64;  // 8 x 8 threads, each a 4 x 4 block of outputs {ti + 8a} x {tj + 8b}
#ifndef CT_MINB
#define CT_MINB 8
#endif
#ifndef CT_UNROLL
#define CT_UNROLL 2
#endif
constexpr int CT_UNROLL_N = CT_UNROLL;

// partial[(c*T + t)*n*n + i*n + j] = sum over k-chunk c of conj(eta_i[k]) g5(k) X_j[k]
// Two-stage cp.async pipeline: the 16-byte copies of stage s+1 (global -> shared, no registers) are in flight while stage s
// is multiplied.  Shared tiles are stored [row][k] with a row stride of 17 x 16 bytes: the copies are coalesced along k
// (a half-warp moves 256 contiguous bytes of one row) and the compute-phase reads of 8 different rows at one k fall in 8
// different bank groups (lanes sharing ti get a broadcast).  conj() and the gamma5 sign are applied when the tile is read back from shared memory.
__global__ void __launch_bounds__(CT_THREADS, CT_MINB) contract_kernel(const double2 *__restrict__ eta, const double2 *__restrict__ xs, int n, int T,
                                                                 long K, long kchunk, int tiles, double2 *__restrict__ partial)
{
    __shared__ __align__(16) double2 As[2][CT_TILE][CT_KT + 1], Bs[2][CT_TILE][CT_KT + 1];
    const int c = blockIdx.x, t = blockIdx.y, bi = blockIdx.z / tiles, bj = blockIdx.z % tiles;
    const int ti = threadIdx.x >> 3, tj = threadIdx.x & 7;
    const long k0 = (long)c * kchunk, k1 = min(K, k0 + kchunk);
    double2 acc[4][4];
#pragma unroll
    for (int a = 0; a < 4; a++)
#pragma unroll
        for (int b = 0; b < 4; b++) acc[a][b] = make_double2(0., 0.);

    auto issue = [&](int stage, long kb) {
        // 32 rows x 16 k per operand; a half-warp copies 256 contiguous bytes of one row (coalesced), 8 copies per thread
#pragma unroll
        for (int it = 0; it < 8; it++) {
            const int item = threadIdx.x + CT_THREADS * it, row = item >> 4, kq = item & 15;
            const long k = kb + kq;
            const int i = bi * CT_TILE + row, j = bj * CT_TILE + row;
            double2 *da = &As[stage][row][kq], *db = &Bs[stage][row][kq];
            if (k < k1 && i < n) __pipeline_memcpy_async(da, eta + ((long)i * T + t) * K + k, 16);
            else *da = make_double2(0., 0.);
            if (k < k1 && j < n) __pipeline_memcpy_async(db, xs + ((long)j * T + t) * K + k, 16);
            else *db = make_double2(0., 0.);
        }
        __pipeline_commit();
    };

    issue(0, k0);
    int stage = 0;
    for (long kb = k0; kb < k1; kb += CT_KT, stage ^= 1) {
        if (kb + CT_KT < k1) {
            issue(stage ^ 1, kb + CT_KT);
            __pipeline_wait_prior(1);
        } else __pipeline_wait_prior(0);
        __syncthreads();
#pragma unroll CT_UNROLL_N
        for (int kk = 0; kk < CT_KT; kk++) {
            const double sgn = (((kb + kk) % 12) < 6) ? 1.0 : -1.0;   // gamma5 = diag(+,+,-,-), spin = (k % 12) / 3
            double2 a[4], b[4];
#pragma unroll
            for (int r = 0; r < 4; r++) {
                const double2 e = As[stage][ti + 8 * r][kk];
                a[r] = make_double2(sgn * e.x, -sgn * e.y);          // conj(eta) gamma5
                b[r] = Bs[stage][tj + 8 * r][kk];
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
    double2 *out = partial + ((long)c * T + t) * n * n;
#pragma unroll
    for (int a = 0; a < 4; a++)
#pragma unroll
        for (int b = 0; b < 4; b++) {
            const int i = bi * CT_TILE + ti + 8 * a, j = bj * CT_TILE + tj + 8 * b;
            if (i < n && j < n) out[(long)i * n + j] = acc[a][b];
        }
}

// O[idx] = sum_c partial[c][idx], fixed order (deterministic)
__global__ void contract_reduce_kernel(const double2 *__restrict__ partial, long count, int nchunks, double2 *__restrict__ o)
{
    const long idx = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= count) return;
    double2 s = make_double2(0., 0.);
    for (int c = 0; c < nchunks; c++) {
        const double2 v = partial[(long)c * count + idx];
        s.x += v.x;
        s.y += v.y;
    }
    o[idx] = s;
}

// C[t0][t] = norm * sum_ij O[t][i][j] O[t0][j][i]
__global__ void __launch_bounds__(256) correlator_kernel(const double2 *__restrict__ o, int n, double norm, double2 *__restrict__ cout)
{
    __shared__ double sre[256], sim[256];
    const int t = blockIdx.x, t0 = blockIdx.y, T = gridDim.x;
    const double2 *ot = o + (long)t * n * n, *o0 = o + (long)t0 * n * n;
    double re = 0, im = 0;
    for (int p = threadIdx.x; p < n * n; p += 256) {
        const int i = p / n, j = p % n;
        const double2 a = ot[p], b = o0[(long)j * n + i];
        re += a.x * b.x - a.y * b.y;
        im += a.x * b.y + a.y * b.x;
    }
    sre[threadIdx.x] = re;
    sim[threadIdx.x] = im;
    __syncthreads();
    for (int s = 128; s > 0; s >>= 1) {
        if ((int)threadIdx.x < s) { sre[threadIdx.x] += sre[threadIdx.x + s]; sim[threadIdx.x] += sim[threadIdx.x + s]; }
        __syncthreads();
    }
    if (threadIdx.x == 0) cout[(long)t0 * T + t] = make_double2(norm * sre[0], norm * sim[0]);
}

int launch_contract(const double *eta, const double *xs, const int dims[4], int n, double *o, cudaStream_t st)
{
    const int T = dims[3];
    const long K = 12L * dims[0] * dims[1] * dims[2];
    const int tiles = (n + CT_TILE - 1) / CT_TILE;
    // enough k-chunks for ~16 CTAs of 64 threads per SM, each chunk a multiple of the staging width
    long nch = std::max<long>(1, (16L * 148 + (long)T * tiles * tiles - 1) / ((long)T * tiles * tiles));
    nch = std::min<long>(nch, std::max<long>(1, K / (8 * CT_KT)));
    long kchunk = (K + nch - 1) / nch;
    kchunk = (kchunk + CT_KT - 1) / CT_KT * CT_KT;
    nch = (K + kchunk - 1) / kchunk;
    const long count = (long)T * n * n;
    double2 *partial = nullptr;
    CLV_CUDA(cudaMallocAsync((void **)&partial, sizeof(double2) * count * nch, st));
    contract_kernel<<<dim3((unsigned)nch, T, tiles * tiles), CT_THREADS, 0, st>>>((const double2 *)eta, (const double2 *)xs, n, T, K, kchunk, tiles, partial);
    CLV_CUDA(cudaGetLastError());
    contract_reduce_kernel<<<(unsigned)((count + 255) / 256), 256, 0, st>>>(partial, count, (int)nch, (double2 *)o);
    CLV_CUDA(cudaGetLastError());
    CLV_CUDA(cudaFreeAsync(partial, st));
    return 0;
}

int launch_correlator(const double *o, int T, int n, double scale, double *c, cudaStream_t st)
{
    const double norm = 1.0 / ((double)n * n * scale * scale * scale * scale);
    correlator_kernel<<<dim3(T, T), 256, 0, st>>>((const double2 *)o, n, norm, (double2 *)c);
    CLV_CUDA(cudaGetLastError());
    return 0;
}

}  // namespace clv
