// noise.cu -- Z4 noise sources, written from docs/NOISE.md ("random source vector", L355 time dilution).
// Pure write stream: 2 complex numbers per thread, canonical layout [rhs][t][z][y][x][spin][colour].
#include "context.h"

namespace clv {

__device__ __forceinline__ unsigned z4_index(uint64_t seed, uint64_t ctr)
{
    uint64_t z = seed + 0x9E3779B97F4A7C15ULL * (ctr + 1ULL);
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
    z ^= z >> 31;
    return (unsigned)(z >> 62);
}

template <typename R> struct Pair;
template <> struct Pair<float> { typedef float4 T; };
template <> struct Pair<double> { typedef double4 T; };

// value table: k -> (re, im) chosen among {+scale, -scale, +0}
template <typename R> __device__ __forceinline__ void z4_value(unsigned k, R scale, R &re, R &im)
{
    const R zero = (R)0;
    re = (k == 0) ? scale : (k == 2) ? -scale : zero;
    im = (k == 1) ? scale : (k == 3) ? -scale : zero;
}

template <typename R>
__global__ void __launch_bounds__(256) noise_kernel(R *__restrict__ out, uint64_t n12V, uint64_t sites_per_t, int T, uint64_t seed, int n_rhs,
                                                    int rhs_offset, int dilution, R scale)
{
    const uint64_t pairs_per_rhs = n12V / 2;
    const bool aligned32 = (reinterpret_cast<uintptr_t>(out) & 31u) == 0;
    const uint64_t total = pairs_per_rhs * (uint64_t)n_rhs;
    for (uint64_t i = (uint64_t)blockIdx.x * 256 + threadIdx.x; i < total; i += (uint64_t)gridDim.x * 256) {
        const uint64_t j = i / pairs_per_rhs, n = 2 * (i % pairs_per_rhs);
        const uint64_t r = (uint64_t)rhs_offset + j;
        R v[4];
        // dilution: bit 0 keeps timeslice r mod T only, bit 1 keeps spin-colour component (r / T or r) mod 12 only (docs/NOISE.md)
        const bool keep_t = !(dilution & 1) || (int)((n / 12) / sites_per_t) == (int)(r % (uint64_t)T);  // n and n+1 share a site
        const int sc_r = (dilution & 2) ? (int)(((dilution & 1) ? r / (uint64_t)T : r) % 12ULL) : -1;
        const int sc0 = (int)(n % 12);
        v[0] = v[1] = v[2] = v[3] = (R)0;
        if (keep_t && (sc_r < 0 || sc_r == sc0)) z4_value<R>(z4_index(seed, r * n12V + n), scale, v[0], v[1]);
        if (keep_t && (sc_r < 0 || sc_r == sc0 + 1)) z4_value<R>(z4_index(seed, r * n12V + n + 1), scale, v[2], v[3]);
        R *dst = out + (j * n12V + n) * 2;
        if (sizeof(R) == 4) {
            *reinterpret_cast<float4 *>(dst) = make_float4((float)v[0], (float)v[1], (float)v[2], (float)v[3]);
        } else if (aligned32) {  // one 32-byte store per thread: a warp writes 1 KB contiguous
            asm volatile("st.global.v4.f64 [%0], {%1,%2,%3,%4};" ::"l"(dst), "d"((double)v[0]), "d"((double)v[1]), "d"((double)v[2]), "d"((double)v[3])
                         : "memory");
        } else {
            *reinterpret_cast<double2 *>(dst) = make_double2((double)v[0], (double)v[1]);
            *reinterpret_cast<double2 *>(dst + 2) = make_double2((double)v[2], (double)v[3]);
        }
    }
}

int launch_noise(void *out, int precision, const int dims[4], uint64_t seed, int n_rhs, int rhs_offset, int dilution, double scale, cudaStream_t st)
{
    const uint64_t V = (uint64_t)dims[0] * dims[1] * dims[2] * dims[3];
    const uint64_t n12V = 12 * V, spt = (uint64_t)dims[0] * dims[1] * dims[2];
    const uint64_t total = n12V / 2 * (uint64_t)n_rhs;
    if (total == 0) return 0;
    const unsigned grid = (unsigned)std::min<uint64_t>((total + 255) / 256, 148u * 64u);
    if (precision == 32) noise_kernel<float><<<grid, 256, 0, st>>>((float *)out, n12V, spt, dims[3], seed, n_rhs, rhs_offset, dilution, (float)scale);
    else noise_kernel<double><<<grid, 256, 0, st>>>((double *)out, n12V, spt, dims[3], seed, n_rhs, rhs_offset, dilution, scale);
    CLV_CUDA(cudaGetLastError());
    return 0;
}

}  // namespace clv
