// common.cuh -- types, internal layout and small device helpers shared by the CUDA translation units.
//
// Internal ("lane-blocked", even-odd) layout, see DESIGN.md sec. 3:
//   site of parity p = (x+y+z+t)&1 has checkerboard index cb = lex/2, lex = ((t*Z+z)*Y+y)*X+x.
//   A spinor field of B right-hand sides on one parity is addressed by j = cb*B + rhs and stored as
//   16-byte vectors  vec[((j>>5)*NV + k)*32 + (j&31)],  k = 0..NV-1:
//     fp32: NV = 6,  vector k = float4  = complex numbers 2k, 2k+1 of the 12 (index 3*spin+colour)
//     fp64: NV = 12, vector k = double2 = complex number k
//   so 32 consecutive j (a warp) read 512 contiguous bytes per k, and the 8 rhs of a site at B = 8 fill
//   one 128-byte line.  Links and clover blocks use the same blocking over cb with complex (Real2)
//   elements:  elem[((cb>>5)*NK + k)*32 + (cb&31)].
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace clv {

template <typename R> struct Vec;
template <> struct Vec<float> { typedef float4 T; typedef float2 C; static constexpr int NV = 6; };
template <> struct Vec<double> { typedef double2 T; typedef double2 C; static constexpr int NV = 12; };

template <typename R> struct cx {
    R re, im;
};

template <typename R> __host__ __device__ __forceinline__ cx<R> mk(R re, R im)
{
    cx<R> c;
    c.re = re;
    c.im = im;
    return c;
}
template <typename R> __host__ __device__ __forceinline__ cx<R> operator+(cx<R> a, cx<R> b) { return mk<R>(a.re + b.re, a.im + b.im); }
template <typename R> __host__ __device__ __forceinline__ cx<R> operator-(cx<R> a, cx<R> b) { return mk<R>(a.re - b.re, a.im - b.im); }
template <typename R> __host__ __device__ __forceinline__ cx<R> operator*(cx<R> a, cx<R> b)
{
    return mk<R>(a.re * b.re - a.im * b.im, a.re * b.im + a.im * b.re);
}
template <typename R> __host__ __device__ __forceinline__ cx<R> operator*(R s, cx<R> a) { return mk<R>(s * a.re, s * a.im); }
template <typename R> __host__ __device__ __forceinline__ cx<R> conj(cx<R> a) { return mk<R>(a.re, -a.im); }
// a + i b, a - i b
template <typename R> __host__ __device__ __forceinline__ cx<R> add_i(cx<R> a, cx<R> b) { return mk<R>(a.re - b.im, a.im + b.re); }
template <typename R> __host__ __device__ __forceinline__ cx<R> sub_i(cx<R> a, cx<R> b) { return mk<R>(a.re + b.im, a.im - b.re); }
// acc += a*b ; acc += conj(a)*b
template <typename R> __host__ __device__ __forceinline__ void fma_cx(cx<R> &acc, cx<R> a, cx<R> b)
{
    acc.re += a.re * b.re;
    acc.re -= a.im * b.im;
    acc.im += a.re * b.im;
    acc.im += a.im * b.re;
}
template <typename R> __host__ __device__ __forceinline__ void fma_conj(cx<R> &acc, cx<R> a, cx<R> b)
{
    acc.re += a.re * b.re;
    acc.re += a.im * b.im;
    acc.im += a.re * b.im;
    acc.im -= a.im * b.re;
}

// ---- lattice geometry (host + device) ---------------------------------------------------------
struct Geom {
    int X, Y, Z, T;    // extents
    int Xh;            // X/2
    int Vh;            // sites per parity
    int bc[4];         // +1 | -1
};

// vector index of (j, k) in a lane-blocked field with NK vectors per entry
__host__ __device__ __forceinline__ unsigned lb_index(unsigned j, int k, int NK) { return ((j >> 5) * NK + k) * 32u + (j & 31u); }
// index (in complex elements) of complex element k of entry cb in a lane-blocked complex field with NK elements per entry.
// fp64: one double2 per (k, lane).  fp32: elements are packed in pairs so that a thread fetches two of them with one
// 16-byte load: per 32-entry block, NK/2 float4 rows [k/2][lane] followed, if NK is odd, by one float2 row [lane].
template <typename R> __host__ __device__ __forceinline__ unsigned cplx_index(unsigned cb, int k, int NK)
{
    if (sizeof(R) == 8) return lb_index(cb, k, NK);
    const unsigned base = (cb >> 5) * 32u * NK, lane = cb & 31u;
    const int n4 = NK / 2;
    return (k < 2 * n4) ? base + ((unsigned)(k >> 1) * 32u + lane) * 2u + (k & 1) : base + (unsigned)n4 * 64u + lane;
}

// number of 32-lane blocks needed for n entries
__host__ __device__ __forceinline__ unsigned lb_blocks(unsigned n) { return (n + 31u) >> 5; }

struct Coord {
    int xh, x, y, z, t;
};

// decode checkerboard index of a site of parity p
__device__ __forceinline__ Coord decode(const Geom &g, int cb, int p)
{
    Coord c;
    c.xh = cb % g.Xh;
    int r = cb / g.Xh;
    c.y = r % g.Y;
    r /= g.Y;
    c.z = r % g.Z;
    c.t = r / g.Z;
    c.x = 2 * c.xh + ((c.y + c.z + c.t + p) & 1);
    return c;
}

// checkerboard index (within the opposite parity) of the neighbour of (cb, c) in direction MU, FWD ? +1 : -1;
// `wrap` tells whether the hop crossed the lattice boundary.
template <int MU, int FWD> __device__ __forceinline__ int neighbour(const Geom &g, int cb, const Coord &c, bool &wrap)
{
    if (MU == 0) {
        const int odd = c.x & 1;
        if (FWD) {
            wrap = (c.x == g.X - 1);
            return wrap ? cb - (g.Xh - 1) : cb + odd;
        } else {
            wrap = (c.x == 0);
            return wrap ? cb + (g.Xh - 1) : cb - (1 - odd);
        }
    } else if (MU == 1) {
        const int s = g.Xh;
        if (FWD) { wrap = (c.y == g.Y - 1); return wrap ? cb - s * (g.Y - 1) : cb + s; }
        else     { wrap = (c.y == 0);       return wrap ? cb + s * (g.Y - 1) : cb - s; }
    } else if (MU == 2) {
        const int s = g.Xh * g.Y;
        if (FWD) { wrap = (c.z == g.Z - 1); return wrap ? cb - s * (g.Z - 1) : cb + s; }
        else     { wrap = (c.z == 0);       return wrap ? cb + s * (g.Z - 1) : cb - s; }
    } else {
        const int s = g.Xh * g.Y * g.Z;
        if (FWD) { wrap = (c.t == g.T - 1); return wrap ? cb - s * (g.T - 1) : cb + s; }
        else     { wrap = (c.t == 0);       return wrap ? cb + s * (g.T - 1) : cb - s; }
    }
}

// ---- spinor / link / clover loads -------------------------------------------------------------
__device__ __forceinline__ void load_spinor(const float4 *__restrict__ f, unsigned j, cx<float> psi[12])
{
    const float4 *p = f + lb_index(j, 0, 6);
#pragma unroll
    for (int k = 0; k < 6; k++) {
        float4 v = __ldg(p + 32 * k);
        psi[2 * k] = mk<float>(v.x, v.y);
        psi[2 * k + 1] = mk<float>(v.z, v.w);
    }
}
__device__ __forceinline__ void load_spinor(const double2 *__restrict__ f, unsigned j, cx<double> psi[12])
{
    const double2 *p = f + lb_index(j, 0, 12);
#pragma unroll
    for (int k = 0; k < 12; k++) {
        double2 v = __ldg(p + 32 * k);
        psi[k] = mk<double>(v.x, v.y);
    }
}
__device__ __forceinline__ void store_spinor(float4 *__restrict__ f, unsigned j, const cx<float> psi[12])
{
    float4 *p = f + lb_index(j, 0, 6);
#pragma unroll
    for (int k = 0; k < 6; k++) p[32 * k] = make_float4(psi[2 * k].re, psi[2 * k].im, psi[2 * k + 1].re, psi[2 * k + 1].im);
}
__device__ __forceinline__ void store_spinor(double2 *__restrict__ f, unsigned j, const cx<double> psi[12])
{
    double2 *p = f + lb_index(j, 0, 12);
#pragma unroll
    for (int k = 0; k < 12; k++) p[32 * k] = make_double2(psi[k].re, psi[k].im);
}

// link at cb: RECON = 18 -> 9 stored complex; RECON = 12 -> rows 0,1 stored, row 2 = conj(row0 x row1) rebuilt by third_row()
// at the point of use (not at the load, so that loads can be issued a direction ahead)
template <typename R, int RECON> __device__ __forceinline__ void third_row(cx<R> u[9])
{
    if (RECON == 12) {
        u[6] = conj(u[1] * u[5] - u[2] * u[4]);
        u[7] = conj(u[2] * u[3] - u[0] * u[5]);
        u[8] = conj(u[0] * u[4] - u[1] * u[3]);
    }
}
template <int RECON> __device__ __forceinline__ void load_link(const double2 *__restrict__ f, unsigned cb, cx<double> u[9])
{
    constexpr int NK = RECON / 2;
    const double2 *p = f + lb_index(cb, 0, NK);
#pragma unroll
    for (int k = 0; k < NK; k++) {
        double2 v = __ldg(p + 32 * k);
        u[k] = mk<double>(v.x, v.y);
    }
}
template <int RECON> __device__ __forceinline__ void load_link(const float2 *__restrict__ f, unsigned cb, cx<float> u[9])
{
    constexpr int NK = RECON / 2, N4 = NK / 2;
    const float2 *blk = f + (cb >> 5) * 32u * NK;
    const unsigned lane = cb & 31u;
    const float4 *p4 = reinterpret_cast<const float4 *>(blk) + lane;
#pragma unroll
    for (int k = 0; k < N4; k++) {
        float4 v = __ldg(p4 + 32 * k);
        u[2 * k] = mk<float>(v.x, v.y);
        u[2 * k + 1] = mk<float>(v.z, v.w);
    }
    if (NK & 1) {
        float2 v = __ldg(blk + N4 * 64 + lane);
        u[NK - 1] = mk<float>(v.x, v.y);
    }
}

// ---- error plumbing (host) ---------------------------------------------------------------------
void set_error(const char *fmt, ...);
#define CLV_CUDA(call)                                                                              \
    do {                                                                                            \
        cudaError_t e_ = (call);                                                                    \
        if (e_ != cudaSuccess) {                                                                    \
            clv::set_error("%s failed at %s:%d: %s", #call, __FILE__, __LINE__, cudaGetErrorString(e_)); \
            return (e_ == cudaErrorMemoryAllocation) ? CLOVER_ENOMEM : CLOVER_ECUDA;                \
        }                                                                                           \
    } while (0)
#define CLV_CHECK(expr)                                                                             \
    do {                                                                                            \
        int rc_ = (expr);                                                                           \
        if (rc_ < 0) return rc_;                                                                    \
    } while (0)

}  // namespace clv
