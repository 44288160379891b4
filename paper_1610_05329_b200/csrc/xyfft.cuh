// xyfft.cuh -- K2, K3, K4 for the specialised line lengths: the FFT passes of the half-spectrum along
// the strided axes y and x (SV section 8a rows a2-a4; BJ:north_star "mixed-radix shared-memory Stockham
// FFT passes per axis", "Udd(k) multiply fused into the forward-last and inverse-first passes").
//
// A tile is 8 neighbouring lines x the whole line, [N][8] complex doubles in shared memory (one row =
// 128 bytes = one L2 line, so every global access of a strided axis is a full line and every
// shared-memory access of a quarter-warp is one conflict-free 128-byte row).  N is a template constant:
// thread (c = tid & 7, b = tid >> 3) keeps the N/NBF elements of its butterflies in registers, the first
// pass reads global memory straight into them, the last pass writes global memory straight from them,
// and only the exchanges between passes go through the tile.
//   K2/K4 (FFT_FWD / FFT_INV): npass-1 exchanges.
//   K3 (FFT_X_UDD): forward transform in the radix order 8,..,3, inverse in the reversed order, so the
//   last forward pass, the Udd~(k)/N multiply and the first inverse pass run on the same registers:
//   2 (npass-1) exchanges for the two transforms.
// Several CTAs are resident per SM (<= 64 registers per thread), so the load, exchange and store
// phases of different tiles overlap.
#pragma once
#include "ctfft.cuh"

namespace dgpe {

struct UddArgs {
    int nzh;                          // kz bins per row of the half-spectrum
    const double *kx2, *ky2, *kz2;    // squared wave numbers (R#10, R#11)
    double dkx;                       // 2 pi/(nx dx): kx of bin m is (m <= nx/2 ? m : m - nx) dkx
    double invN;                      // 1/(nx ny nz): normalisation of the inverse transform (R#10)
    int pf_tiles;                     // L2 prefetch distance in tiles (one residency of CTAs); 0 = off
};

enum { FFT_FWD = 0, FFT_INV = 1, FFT_X_UDD = 2 };

struct PosTile {
    static __device__ __forceinline__ int at(int idx) { return idx * TILE_COLS; }
};

template <int N>
__host__ __device__ constexpr int xy_nbf() { return N / ct::rmax(N); }
template <int N>
__host__ __device__ constexpr int xy_threads() { return (TILE_COLS * xy_nbf<N>() + 31) / 32 * 32; }
// CTAs per SM the register budget is tuned for: 64 registers per thread, bounded by shared memory
template <int N>
__host__ __device__ constexpr int xy_min_ctas()
{
    int by_regs = 65536 / (64 * xy_threads<N>());
    int by_smem = (227 * 1024) / (N * TILE_COLS * 16);
    int m = by_regs < by_smem ? by_regs : by_smem;
    return m < 1 ? 1 : (m > 8 ? 8 : m);
}

// grid = (ceil(ncols/8), nbatch); block = xy_threads<N>(); dynamic shared memory = N*128 bytes.
template <int N, int KIND>
__global__ void __launch_bounds__(xy_threads<N>(), xy_min_ctas<N>())
k_fft_xy(cplx* __restrict__ data, LineMap map, const cplx* __restrict__ tw, UddArgs U)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    constexpr int NBF = xy_nbf<N>();
    constexpr int L = ct::npass(N);
    const int tid = threadIdx.x, c = tid & 7, b = tid >> 3;
    const int col = blockIdx.x * TILE_COLS + c;
    const bool colok = col < map.ncols;
    const bool on = colok && b < NBF;
    cplx* g = data + (long long)blockIdx.y * map.batch_stride + (long long)(colok ? col : 0) * map.col_stride;
    const long long es = map.elem_stride;
    cplx* colsm = reinterpret_cast<cplx*>(smem_raw) + c;
    if (U.pf_tiles > 0) {
        // ask L2 for the tile a CTA will process one residency later (rows of 128 bytes, which straddle
        // two lines when the half-spectrum row length nz/2+1 is odd)
        const long long id = (long long)blockIdx.y * gridDim.x + blockIdx.x + U.pf_tiles;
        const int by = (int)(id / gridDim.x), bx = (int)(id - (long long)by * gridDim.x);
        if (by < (int)gridDim.y) {
            const char* t0 = reinterpret_cast<const char*>(data + (long long)by * map.batch_stride +
                                                           (long long)bx * TILE_COLS * map.col_stride);
            for (int j = tid; j < 2 * N; j += xy_threads<N>())
                prefetch_l2(t0 + (long long)(j >> 1) * es * 16 + (j & 1) * 112);
        }
    }
    auto from_g = [&](int idx) { return ld_stream(g + (long long)idx * es); };
    auto to_g = [&](int idx, cplx v) { st_stream(g + (long long)idx * es, v); };

    if constexpr (KIND != FFT_X_UDD) {
        ct_fft_range<N, KIND == FFT_INV, false, NBF, SyncCta, PosTile, 0, L, true>(colsm, b, on, tw, from_g, to_g);
    } else {
        // ky^2, kz^2 of this thread's column, loaded now and used after the forward passes
        const int ky = (colok ? col : 0) / U.nzh, kz = (colok ? col : 0) - ky * U.nzh;
        const double qy = __ldg(&U.ky2[ky]), qz = __ldg(&U.kz2[kz]);
        // forward passes 0 .. L-2 through the tile
        ct_fft_range<N, false, false, NBF, SyncCta, PosTile, 0, L - 1, true>(colsm, b, on, tw, from_g, to_g);
        // last forward pass, Udd~(k)/N, first inverse pass: one set of registers
        using PF = CtPass<N, L - 1, false, false, NBF>;
        using PI = CtPass<N, 0, true, true, NBF>;
        static_assert(PF::R == PI::R && PF::NB == PI::NB && PI::Ns == 1, "forward-last and inverse-first passes must match");
        PF pf;
        if (on) {
            pf.load_tw(b, tw);
            if constexpr (L == 1) pf.load(b, from_g);
            else pf.load(b, [&](int idx) { return colsm[PosTile::at(idx)]; });
        }
        if constexpr (L > 1) __syncthreads();
        PI pi;
        if (on) {
            pf.bfly(b);
            // Udd~(k) = (4 pi/3)(3 kz^2/|k|^2 - 1), Udd~(0) = 0 (BJ:configs[0]; R#11); column = (ky, kz) flattened
            const double FOUR_PI_3 = 4.1887902047863909846168578443727;
            pf.modify(b, [&](int idx, cplx v) {
                // kx^2 from the bin index (f = idx or idx - N, R#10) instead of a table load whose latency
                // would sit in the middle of the register chain
                const double kx = (double)(idx <= N / 2 ? idx : idx - N) * U.dkx;
                const double k2 = kx * kx + qy + qz;
                // 1/k2 by two Newton steps from the single-precision reciprocal (<= 2 ulp; k2 is a sum of
                // squared wave numbers, far inside the float range; k2 = 0 gives inf/NaN, replaced below)
                double rk = (double)__frcp_rn((float)k2);
                rk = rk * (2.0 - k2 * rk);
                rk = rk * (2.0 - k2 * rk);
                double u = FOUR_PI_3 * (3.0 * qz * rk - 1.0);
                if (k2 == 0.0) u = 0.0;      // Udd~(0) = 0 (R#11); k2 is exactly zero only at the origin
                u *= U.invN;
                return mk(v.x * u, v.y * u);
            });
#pragma unroll
            for (int u = 0; u < PF::NB; ++u)
#pragma unroll
                for (int q = 0; q < PF::R; ++q) pi.v[u][q] = pf.v[u][q];
            pi.bfly(b);
        }
        if constexpr (L == 1) {
            if (on) pi.scatter(b, to_g);
        } else {
            if (on) pi.scatter(b, [&](int idx, cplx val) { colsm[PosTile::at(idx)] = val; });
            __syncthreads();
            ct_fft_range<N, true, true, NBF, SyncCta, PosTile, 1, L, false>(colsm, b, on, tw, from_g, to_g);
        }
    }
}

}  // namespace dgpe
