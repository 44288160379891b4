// common.cuh -- complex-double helpers, block reductions and shared kernel-argument structs.
// Part of libdgpe (include/dgpe.h).  Shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace dgpe {

typedef double2 cplx;   // (re, im), 16 bytes: one vectorised LDG/STG/LDS/STS.128 per element

constexpr int TILE_COLS = 8;        // 8 complex doubles = 128 bytes: one full L2 line per tile row
constexpr int MAX_PASSES = 10;      // 1024 = 8*8*4*4 needs 4; 3^6 = 729 needs 6
constexpr int MAX_RED = 8;          // values reduced together by one kernel

__device__ __forceinline__ cplx mk(double x, double y) { return make_double2(x, y); }
__device__ __forceinline__ cplx cadd(cplx a, cplx b) { return mk(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ cplx csub(cplx a, cplx b) { return mk(a.x - b.x, a.y - b.y); }
__device__ __forceinline__ cplx cmul(cplx a, cplx b) { return mk(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }
__device__ __forceinline__ cplx cscale(cplx a, double s) { return mk(a.x * s, a.y * s); }
__device__ __forceinline__ cplx cconj(cplx a) { return mk(a.x, -a.y); }
__device__ __forceinline__ cplx mul_pi(cplx a) { return mk(-a.y, a.x); }   // * (+i)
__device__ __forceinline__ cplx mul_mi(cplx a) { return mk(a.y, -a.x); }   // * (-i)
__device__ __forceinline__ double cabs2(cplx a) { return a.x * a.x + a.y * a.y; }

// Coefficient arithmetic of the Crank-Nicolson tables: real in imaginary time, complex in real time.
__device__ __forceinline__ cplx coef_mul(double c, cplx v) { return mk(c * v.x, c * v.y); }
__device__ __forceinline__ cplx coef_mul(cplx c, cplx v) { return cmul(c, v); }
__device__ __forceinline__ double coef_neg(double c) { return -c; }
__device__ __forceinline__ cplx coef_neg(cplx c) { return mk(-c.x, -c.y); }
// a + c*b
__device__ __forceinline__ cplx coef_fma(double c, cplx b, cplx a) { return mk(fma(c, b.x, a.x), fma(c, b.y, a.y)); }
__device__ __forceinline__ cplx coef_fma(cplx c, cplx b, cplx a)
{
    return mk(fma(c.x, b.x, fma(-c.y, b.y, a.x)), fma(c.x, b.y, fma(c.y, b.x, a.y)));
}

// Right-hand side of one Crank-Nicolson line equation, d_j = r p_{j-1} + (1 - 2r) p_j + r p_{j+1} (R#9).
// Imaginary time: r real.  Real time: r = i rho is purely imaginary (r = i dt/(4 d^2)), so
// d_j = p_j + i rho (p_{j-1} + p_{j+1} - 2 p_j): 6 operations instead of the 10 of two general complex products.
__device__ __forceinline__ cplx cn_rhs(double r, double omr2, cplx a, cplx m, cplx b)
{
    return coef_fma(omr2, m, coef_mul(r, cadd(a, b)));
}
__device__ __forceinline__ double cn_rhs(double r, double omr2, double a, double m, double b)
{
    return fma(omr2, m, r * (a + b));
}
__device__ __forceinline__ cplx cn_rhs(cplx r, cplx /*omr2*/, cplx a, cplx m, cplx b)
{
    const double sx = fma(-2.0, m.x, a.x + b.x), sy = fma(-2.0, m.y, a.y + b.y);
    return mk(fma(-r.y, sy, m.x), fma(r.y, sx, m.y));
}

// sin x and cos x for the real-time exponential exp(-i dt H) (BJ:north_star (b)), branch-free: two-constant
// Cody-Waite reduction r = x - k pi/2 (k = rint(2x/pi); both products exact inside the fmas) and the Taylor
// polynomials of sin and cos on |r| <= pi/4 (truncation 4.6e-17 and 2e-18).  Absolute error <= 2e-16 for
// |x| < SINCOS_FAST_LIMIT = 2^30 (the reduction itself holds far beyond; the limit is where the caller switches
// to the library routine, which is exact for any double).  NaN and inf give NaN, as the library's does.
constexpr double SINCOS_FAST_LIMIT = 1073741824.0;
__device__ __forceinline__ void sincos_fast(double x, double* sn, double* cs)
{
    const double t = fma(x, 0.63661977236758134308, 6755399441055744.0);      // 2/pi; 1.5 * 2^52: rint in the low bits
    const int q = __double2loint(t);
    const double k = t - 6755399441055744.0;
    double r = fma(-k, 1.57079632679489655800e+00, x);                          // pi/2, high part
    r = fma(-k, 6.12323399573676603587e-17, r);                                 // pi/2, low part
    const double r2 = r * r;
    double ps = -1.0 / 1307674368000.0;                                         // -1/15!
    ps = fma(ps, r2, 1.0 / 6227020800.0);
    ps = fma(ps, r2, -1.0 / 39916800.0);
    ps = fma(ps, r2, 1.0 / 362880.0);
    ps = fma(ps, r2, -1.0 / 5040.0);
    ps = fma(ps, r2, 1.0 / 120.0);
    ps = fma(ps, r2, -1.0 / 6.0);
    const double s = fma(r * r2, ps, r);
    double pc = 1.0 / 20922789888000.0;                                         // 1/16!
    pc = fma(pc, r2, -1.0 / 87178291200.0);
    pc = fma(pc, r2, 1.0 / 479001600.0);
    pc = fma(pc, r2, -1.0 / 3628800.0);
    pc = fma(pc, r2, 1.0 / 40320.0);
    pc = fma(pc, r2, -1.0 / 720.0);
    pc = fma(pc, r2, 1.0 / 24.0);
    pc = fma(pc, r2, -0.5);
    const double c = fma(pc, r2, 1.0);
    // quadrant k mod 4: (s, c), (c, -s), (-s, -c), (-c, s)
    const double a = (q & 1) ? c : s, b = (q & 1) ? s : c;
    *sn = (q & 2) ? -a : a;
    *cs = ((q + 1) & 2) ? -b : b;
}

// Real-valued psi (imaginary time, SV section 8f NEXT-2): the same sweep arithmetic on plain doubles.
__device__ __forceinline__ double cadd(double a, double b) { return a + b; }
__device__ __forceinline__ double csub(double a, double b) { return a - b; }
__device__ __forceinline__ double cabs2(double a) { return a * a; }
__device__ __forceinline__ double coef_mul(double c, double v) { return c * v; }
__device__ __forceinline__ double coef_fma(double c, double b, double a) { return fma(c, b, a); }
// p ? a : b, per component
__device__ __forceinline__ double el_sel(bool p, double a, double b) { return p ? a : b; }
__device__ __forceinline__ cplx el_sel(bool p, cplx a, cplx b) { return mk(p ? a.x : b.x, p ? a.y : b.y); }

// Mixed-radix plan of one 1-D transform length (built on the host in dgpe_api.cu).
struct FftPlan {
    int n;                    // transform length
    int npass;                // number of Stockham passes
    int nbf;                  // butterfly threads per tile column  (= n / largest radix)
    int radix[MAX_PASSES];    // radix of pass p  (2, 3, 4 or 8)
    int nb[MAX_PASSES];       // butterflies each thread holds in registers in pass p
    const cplx* tw;           // tw[j] = exp(-2 pi i j / n), j = 0..n-1 (device)
};

// How a kernel finds the 1-D lines of one axis inside a row-major 3-D array: a "tile" is
// TILE_COLS neighbouring lines; line `col` of batch `bat` has its element j at
//   base[bat*batch_stride + col*col_stride + j*elem_stride].
struct LineMap {
    int n;                  // elements per line
    int ncols;              // lines per batch
    long long batch_stride;
    long long col_stride;
    long long elem_stride;
};

// Deterministic grid-wide sum of NV doubles per thread: warp shuffles, one shared-memory stage, one
// partial per block, and the last block to arrive (atomic ticket) adds the partials in a fixed order.
// Returns true in thread 0 of that last block, with the totals in tot[].
template <int NV>
__device__ __forceinline__ bool grid_reduce(double (&v)[NV], double* partials, unsigned int* ticket,
                                            double (&tot)[NV], double* red /* >= 32*NV doubles smem */)
{
    const int tid = threadIdx.x + blockDim.x * threadIdx.y;
    const int nthr = blockDim.x * blockDim.y;
    const int lane = tid & 31, warp = tid >> 5, nwarp = (nthr + 31) >> 5;
    const unsigned int nblk = gridDim.x * gridDim.y;
    const unsigned int blk = blockIdx.x + gridDim.x * blockIdx.y;
#pragma unroll
    for (int i = 0; i < NV; ++i) {
        double x = v[i];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) x += __shfl_down_sync(0xffffffffu, x, o);
        if (lane == 0) red[warp * NV + i] = x;
    }
    __syncthreads();
    if (warp == 0) {
#pragma unroll
        for (int i = 0; i < NV; ++i) {
            double x = (lane < nwarp) ? red[lane * NV + i] : 0.0;
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) x += __shfl_down_sync(0xffffffffu, x, o);
            if (lane == 0) partials[(size_t)blk * NV + i] = x;
        }
    }
    __shared__ bool is_last;
    if (tid == 0) {
        __threadfence();
        unsigned int t = atomicAdd(ticket, 1u);
        is_last = (t == nblk - 1);
    }
    __syncthreads();
    if (!is_last) return false;
    __threadfence();
    // last block: thread t adds partials t, t+nthr, ... ; then the same two-stage tree
    double acc[NV];
#pragma unroll
    for (int i = 0; i < NV; ++i) acc[i] = 0.0;
    for (unsigned int b = tid; b < nblk; b += nthr) {
#pragma unroll
        for (int i = 0; i < NV; ++i) acc[i] += __ldcg(&partials[(size_t)b * NV + i]);
    }
    __syncthreads();
#pragma unroll
    for (int i = 0; i < NV; ++i) {
        double x = acc[i];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) x += __shfl_down_sync(0xffffffffu, x, o);
        if (lane == 0) red[warp * NV + i] = x;
    }
    __syncthreads();
    bool winner = false;
    if (warp == 0) {
#pragma unroll
        for (int i = 0; i < NV; ++i) {
            double x = (lane < nwarp) ? red[lane * NV + i] : 0.0;
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) x += __shfl_down_sync(0xffffffffu, x, o);
            tot[i] = x;
        }
        if (lane == 0) {
            *ticket = 0u;     // re-arm for the next launch (same stream, so ordered)
            winner = true;
        }
    }
    return winner;
}

// Device scalars carried from step to step (h->scal):
//   [0] s2   = 1/norm of the previous imaginary-time step (density scale),  1 otherwise
//   [1] s1   = 1/sqrt(norm)                               (psi scale),      1 otherwise
//   [2] norm = last norm computed by the folded reduction
//   [3] bad  = 1.0 if any folded norm was not a positive finite number
enum { SC_S2 = 0, SC_S1 = 1, SC_NORM = 2, SC_BAD = 3, SC_COUNT = 8 };

}  // namespace dgpe
