// contract.cu -- stochastic-operator contraction of arXiv:1405.4524, eqs. 7.5-7.7, SURVEY 8(f) rank 1:
//   O_ij(t)   = sum_y eta_i^*(t,y) gamma5 X_j(t,y)            one complex number per (t, i, j)
//   C(t0, t)  = (1/(N_r^2 scale^4)) sum_ij O_ij(t) O_ji(t0)
// Per timeslice this is a complex GEMM  O(t) = conj(E_t) diag(gamma5) X_t^T  with M = N = N_r and K = 12 L^3 (the one dense
// contraction of the paper's pipeline).  The propagators come out of clover_solve in fp64 and parity is asked at 1e-13, so
// the product runs in fp64 on the tensor pipe: tcgen05 has no fp64 type, the fp64 tensor instruction is mma.sync (DMMA, same
// peak as the FMA pipe on B200 at an eighth of the issue slots and register traffic).  At N_r = 32 the arithmetic intensity
// (8 N_r^2 K flop over 32 N_r K bytes = N_r/4 flop/byte) sits at the fp64 ridge of a B200, not above it.
// Canonical layouts: eta, X = [n][T][Z][Y][X][4][3] complex128; O = [T][n][n] complex128; C = [T][T] complex128.
#include "context.h"
#include <algorithm>
#include <cuda_pipeline.h>
#include <mutex>

namespace clv {

constexpr int CT_TILE = 32;    // (i, j) tile edge
constexpr int CT_KT = 16;      // complex k elements staged per step (256 contiguous bytes of every row)
constexpr int CT_KS = CT_KT + 4;   // row stride of the shared tiles in complex numbers: 16 words mod 32, so the two rows of a quarter-warp's 16-byte fragment loads fall in disjoint banks
constexpr int CT_WARPS = 2;    // warp w owns columns [16 w, 16 w + 16) of the tile: 4 x 2 DMMA tiles x 3 accumulator sets
constexpr int CT_THREADS = 32 * CT_WARPS;

// D (8x8, fp64) += A (8x4, row) B (4x8, col): the fp64 tensor-core instruction of sm_80+ (SASS DMMA).  Fragments per thread T:
// a = A[T/4][T%4], b = B[T%4][T/4], c/d = C[T/4][2 (T%4) + {0,1}].
__device__ __forceinline__ void dmma884(double (&c)[2], double a, double b)
{
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};" : "+d"(c[0]), "+d"(c[1]) : "d"(a), "d"(b));
}

// partial[(c*T + t)*n*n + i*n + j] = sum over k-chunk c of conj(eta_i[k]) g5(k) X_j[k]
// Three REAL GEMMs per complex one (Gauss' three-multiplication form, a quarter fewer DMMA than the four-product form): with e = a + i b,
// g5 x = c + i d,   conj(e) x = (ac + bd) + i (ad - bc) = (k1 + k3) + i (k1 + k2),   k1 = (a - b) c,  k2 = a (d - c),  k3 = b (c + d);
// the three sums over k are kept in three accumulator sets and combined once at the end.  Operands are staged [row][k] in shared memory by a
// two-stage cp.async pipeline (16-byte copies, coalesced along k); a 16-byte fragment load brings (a, b) or (c, d) of one (row, k).
__global__ void __launch_bounds__(CT_THREADS) contract_kernel(const double2 *__restrict__ eta, const double2 *__restrict__ xs, int n, int T,
                                                           long K, long kchunk, int tiles, double2 *__restrict__ partial)
{
    __shared__ __align__(16) double2 As[2][CT_TILE][CT_KS], Bs[2][CT_TILE][CT_KS];
    const int c = blockIdx.x, t = blockIdx.y, bi = blockIdx.z / tiles, bj = blockIdx.z % tiles;
    const int w = threadIdx.x >> 5, lane = threadIdx.x & 31, fr = lane >> 2, fk = lane & 3;
    const long k0 = (long)c * kchunk, k1 = min(K, k0 + kchunk);
    double acc1[4][2][2], acc2[4][2][2], acc3[4][2][2];
#pragma unroll
    for (int x = 0; x < 4; x++)
#pragma unroll
        for (int y = 0; y < 2; y++)
#pragma unroll
            for (int e = 0; e < 2; e++) acc1[x][y][e] = acc2[x][y][e] = acc3[x][y][e] = 0.0;

    auto issue = [&](int stage, long kb) {   // 32 rows x 16 k per operand: 16 lanes copy the 256 contiguous bytes of one row
#pragma unroll
        for (int it = 0; it < CT_TILE * CT_KT / CT_THREADS; it++) {
            const int item = threadIdx.x + CT_THREADS * it, row = item / CT_KT, kq = item % CT_KT;
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
    int stage = 0, kbm = (int)(k0 % 12);   // kb mod 12, kept in 32-bit arithmetic (spin-colour index of the block's first element)
    for (long kb = k0; kb < k1; kb += CT_KT, stage ^= 1, kbm = (kbm + CT_KT) % 12) {
        if (kb + CT_KT < k1) {
            issue(stage ^ 1, kb + CT_KT);
            __pipeline_wait_prior(1);
        } else __pipeline_wait_prior(0);
        __syncthreads();
#pragma unroll
        for (int s = 0; s < CT_KT / 4; s++) {   // four complex k per DMMA step; this lane's k = 4 s + fk
            const int sc = kbm + 4 * s + fk;                                     // < 28
            const int scm = sc >= 24 ? sc - 24 : (sc >= 12 ? sc - 12 : sc);
            const double sgn = scm < 6 ? 1.0 : -1.0;                             // gamma5 = diag(+,+,-,-), spin = (k % 12) / 3
            double a[4], b[4], amb[4], cc[2], dmc[2], cpd[2];
#pragma unroll
            for (int r = 0; r < 4; r++) {
                const double2 e = As[stage][8 * r + fr][4 * s + fk];
                a[r] = e.x; b[r] = e.y; amb[r] = e.x - e.y;
            }
#pragma unroll
            for (int r = 0; r < 2; r++) {
                const double2 x = Bs[stage][16 * w + 8 * r + fr][4 * s + fk];
                const double xc = sgn * x.x, xd = sgn * x.y;
                cc[r] = xc; dmc[r] = xd - xc; cpd[r] = xc + xd;
            }
#pragma unroll
            for (int x = 0; x < 4; x++)
#pragma unroll
                for (int y = 0; y < 2; y++) {
                    dmma884(acc1[x][y], amb[x], cc[y]);
                    dmma884(acc2[x][y], a[x], dmc[y]);
                    dmma884(acc3[x][y], b[x], cpd[y]);
                }
        }
        __syncthreads();
    }
    double2 *out = partial + ((long)c * T + t) * n * n;
#pragma unroll
    for (int x = 0; x < 4; x++)
#pragma unroll
        for (int y = 0; y < 2; y++)
#pragma unroll
            for (int e = 0; e < 2; e++) {
                const int i = bi * CT_TILE + 8 * x + fr, j = bj * CT_TILE + 16 * w + 8 * y + 2 * fk + e;
                if (i < n && j < n) out[(long)i * n + j] = make_double2(acc1[x][y][e] + acc3[x][y][e], acc1[x][y][e] + acc2[x][y][e]);
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
    // enough k-chunks for two waves of the CTAs resident on the device (5 per SM), each chunk a multiple of the staging width
    long nch = std::max<long>(1, (10L * 148 + (long)T * tiles * tiles - 1) / ((long)T * tiles * tiles));
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

// ---- allocation-free variant of launch_contract (include/clover.h: stochastic_operators_noalloc) -----------------------------------
// For callers that cannot allocate (code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc): the per-chunk
// partial sums live in this fixed array instead of a cudaMallocAsync block.  Every GPU that loads the library holds its 16 MiB until exit.
// In host code `ct_noalloc_scratch` is only the host-side stand-in of the symbol, NOT a device address: the device address is taken with
// cudaGetSymbolAddress once per device (with that device current) and that pointer is what the kernels get.
// All calls share the array and it keeps the last call's contents.  Nothing in it has to start at zero: every element of the
// [nch][T][n][n] block that contract_reduce_kernel reads is written first by contract_kernel of the same call (every k-chunk is non-empty
// and every (t, tile) CTA stores its whole tile), so no clear is issued.  Two calls that overlap on the GPU (different streams, or two
// host threads) race on the array: callers serialise them.
constexpr long CT_NOALLOC_MAX = 1L << 20;   // complex numbers (CLOVER_NOALLOC_MAX_TNN in clover.h): T * n_rhs^2 * chunks must fit
static __device__ __align__(256) double2 ct_noalloc_scratch[CT_NOALLOC_MAX];

static int noalloc_scratch_ptr(double2 **out)
{
    constexpr int MAX_DEV = 64;
    static std::mutex mu;
    static double2 *ptr[MAX_DEV] = {};
    int dev = -1;
    CLV_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= MAX_DEV) { set_error("stochastic_operators_noalloc: device ordinal %d out of range", dev); return CLOVER_EINVAL; }
    std::lock_guard<std::mutex> lock(mu);
    if (!ptr[dev]) {
        void *q = nullptr;
        CLV_CUDA(cudaGetSymbolAddress(&q, ct_noalloc_scratch));   // device `dev` is current: this is ITS copy of the array
        ptr[dev] = static_cast<double2 *>(q);
    }
    *out = ptr[dev];
    return 0;
}

int launch_contract_noalloc(const double *eta, const double *xs, const int dims[4], int n, double *o, cudaStream_t st)
{
    const int T = dims[3];
    const long K = 12L * dims[0] * dims[1] * dims[2];
    const int tiles = (n + CT_TILE - 1) / CT_TILE;
    const long count = (long)T * n * n;
    if (count > CT_NOALLOC_MAX) {
        set_error("stochastic_operators_noalloc: T * n_rhs^2 = %ld exceeds the fixed scratch of %ld complex numbers (use stochastic_operators)", count,
                  CT_NOALLOC_MAX);
        return CLOVER_EINVAL;
    }
    // k-chunks as in launch_contract, but no more than the scratch holds
    long nch = std::max<long>(1, (10L * 148 + (long)T * tiles * tiles - 1) / ((long)T * tiles * tiles));
    nch = std::min<long>(nch, std::max<long>(1, K / (8 * CT_KT)));
    nch = std::min<long>(nch, CT_NOALLOC_MAX / count);
    long kchunk = (K + nch - 1) / nch;
    kchunk = (kchunk + CT_KT - 1) / CT_KT * CT_KT;
    nch = (K + kchunk - 1) / kchunk;
    double2 *partial = nullptr;
    CLV_CHECK(noalloc_scratch_ptr(&partial));
    contract_kernel<<<dim3((unsigned)nch, T, tiles * tiles), CT_THREADS, 0, st>>>((const double2 *)eta, (const double2 *)xs, n, T, K, kchunk, tiles, partial);
    CLV_CUDA(cudaGetLastError());
    contract_reduce_kernel<<<(unsigned)((count + 255) / 256), 256, 0, st>>>(partial, count, (int)nch, (double2 *)o);
    CLV_CUDA(cudaGetLastError());
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
