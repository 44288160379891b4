// spectral.cuh -- kernels K1..K5 of the step: the dipolar mean field by the
// convolution theorem with a real-to-complex density transform, and the nonlinear /
// potential exponential (BJ:north_star (a), (b)).
//
//   K1 k_dens_r2c     n = s2 |psi|^2, packed two reals per complex, nz/2-point FFT along z, split into
//                     the nz/2+1 Hermitian half-spectrum                       psi (16N) -> spec (S)
//   K2 k_fft_lines    forward FFT along y                                      spec -> spec (2S)
//   K3 k_fft_x_udd    forward FFT along x, multiply by Udd~(k)/N, inverse FFT along x        (2S)
//   K4 k_fft_lines    inverse FFT along y                                                    (2S)
//   K5 k_c2r_nonlin   merge + nz/2-point inverse FFT along z gives Phi; psi <- exp(-dt H) s1 psi or
//                     exp(-i dt H) psi;  or (observe mode) the sums of V n, n^2, Phi n, n
//
// Spectrum layout: spec[i][j][kz], kz = 0..nz/2 contiguous (nzh = nz/2+1 per row), complex double.
#pragma once
#include "fft.cuh"

namespace dgpe {

// ------------------------------------------------------------------------------------------------
// K2 / K4 (and the building block of K3): FFT of the lines described by `map`, in place in global
// memory.  grid = (ceil(ncols/8), nbatch); block = 8*nbf threads (rounded up to a warp multiple);
// dynamic shared memory = n*8*16 bytes.
// ------------------------------------------------------------------------------------------------
template <bool INV, int MAXT>
__global__ void __launch_bounds__(MAXT, 1) k_fft_lines(cplx* __restrict__ data, LineMap map, FftPlan P)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cplx* sm = reinterpret_cast<cplx*>(smem_raw);
    const int c = threadIdx.x & 7, b = threadIdx.x >> 3;
    const int col = blockIdx.x * TILE_COLS + c;
    const bool active = (col < map.ncols) && (b < P.nbf);
    cplx* g = data + (long long)blockIdx.y * map.batch_stride + (long long)col * map.col_stride;
    fft_run<INV>(P, b, active, g, map.elem_stride, sm + c, TILE_COLS, g, map.elem_stride);
}

// ------------------------------------------------------------------------------------------------
// K3: x-pass forward, Udd~(k)/N multiply, x-pass inverse (BJ:north_star "Udd(k) multiply fused into
// the forward-last and inverse-first passes" -- both are the x axis, hence one kernel).
// The columns are the flattened (ky, kz) pairs: col = ky*nzh + kz, element stride ny*nzh.
//   Udd~(k) = (4 pi/3)(3 kz^2/(kx^2+ky^2+kz^2) - 1),  Udd~(0) = 0      (BJ:configs[0]; R#11)
// kx2/ky2/kz2 hold the squared wave numbers k = 2 pi f/(n d), f = m (m <= n/2) or m - n  (R#10).
// invN = 1/(nx ny nz) is the normalisation of the inverse transform (R#10).
// ------------------------------------------------------------------------------------------------
template <int MAXT>
__global__ void __launch_bounds__(MAXT, 1) k_fft_x_udd(cplx* __restrict__ spec, LineMap map, FftPlan P, int nzh,
                            const double* __restrict__ kx2, const double* __restrict__ ky2,
                            const double* __restrict__ kz2, double invN)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cplx* sm = reinterpret_cast<cplx*>(smem_raw);
    const int c = threadIdx.x & 7, b = threadIdx.x >> 3;
    const int col = blockIdx.x * TILE_COLS + c;
    const bool active = (col < map.ncols) && (b < P.nbf);
    cplx* g = spec + (long long)col * map.col_stride;
    const int n = map.n;

    fft_run<false>(P, b, active, g, map.elem_stride, sm + c, TILE_COLS, sm + c, TILE_COLS);

    if (col < map.ncols) {
        const int ky = col / nzh, kz = col - ky * nzh;
        const double qy = __ldg(&ky2[ky]), qz = __ldg(&kz2[kz]);
        const double FOUR_PI_3 = 4.1887902047863909846168578443727;
        for (int i = b; i < n; i += (blockDim.x >> 3)) {
            const double k2 = __ldg(&kx2[i]) + qy + qz;
            double u = 0.0;
            if (k2 != 0.0) u = FOUR_PI_3 * (3.0 * qz / k2 - 1.0);      // k2 is exactly zero only at the origin (R#11)
            u *= invN;
            cplx v = sm[i * TILE_COLS + c];
            sm[i * TILE_COLS + c] = mk(v.x * u, v.y * u);
        }
    }
    __syncthreads();

    fft_run<true>(P, b, active, sm + c, TILE_COLS, sm + c, TILE_COLS, g, map.elem_stride);
}

// ------------------------------------------------------------------------------------------------
// K1: density + real-to-complex transform along z.
// A tile is 8 neighbouring z-lines (line = i*ny + j).  With M = nz/2 the real line n_0..n_{nz-1}
// is packed as z_m = n_{2m} + i n_{2m+1}; Z = DFT_M(z); then for k = 0..M
//   X_k = (Z_k + conj Z_{M-k})/2 - (i/2) e^{-2 pi i k/nz} (Z_k - conj Z_{M-k}),   Z_M := Z_0.
// tws[k] = exp(-2 pi i k/nz), k = 0..M.   scal[SC_S2] scales the density (folded renormalisation).
// grid = ceil(nlines/8); dynamic shared memory = M*8*16 bytes.
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(512, 1) k_dens_r2c(const cplx* __restrict__ psi, cplx* __restrict__ spec, int nlines, int nz,
                           FftPlan P, const cplx* __restrict__ tws, const double* __restrict__ scal)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cplx* sm = reinterpret_cast<cplx*>(smem_raw);
    const int c = threadIdx.x & 7, b = threadIdx.x >> 3, nb = blockDim.x >> 3;
    const int line = blockIdx.x * TILE_COLS + c;
    const bool valid = line < nlines;
    const int M = nz >> 1, nzh = M + 1;
    const double s2 = scal[SC_S2];

    if (valid) {
        const cplx* p = psi + (long long)line * nz;
        for (int m = b; m < M; m += nb) {
            cplx a0 = p[2 * m], a1 = p[2 * m + 1];
            sm[m * TILE_COLS + c] = mk(s2 * cabs2(a0), s2 * cabs2(a1));
        }
    }
    __syncthreads();

    fft_run<false>(P, b, valid && (b < P.nbf), sm + c, TILE_COLS, sm + c, TILE_COLS, sm + c, TILE_COLS);

    if (valid) {
        cplx* out = spec + (long long)line * nzh;
        for (int k = b; k <= M; k += nb) {
            const int k1 = (k == M) ? 0 : k, k2 = (k == 0) ? 0 : M - k;
            cplx zk = sm[k1 * TILE_COLS + c];
            cplx zm = cconj(sm[k2 * TILE_COLS + c]);
            cplx w = __ldg(&tws[k]);
            cplx s = cadd(zk, zm), d = csub(zk, zm);
            cplx wd = cmul(w, d);                       // w (Z_k - conj Z_{M-k})
            // X = s/2 - (i/2) wd  =  ( s.x/2 + wd.y/2 ,  s.y/2 - wd.x/2 )
            out[k] = mk(0.5 * (s.x + wd.y), 0.5 * (s.y - wd.x));
        }
    }
}

// ------------------------------------------------------------------------------------------------
// K5: complex-to-real inverse transform along z, then the nonlinear / potential exponential.
// From the half-spectrum X_0..X_M of one line:
//   Z_k = (X_k + conj X_{M-k}) + i e^{+2 pi i k/nz} (X_k - conj X_{M-k}),   k = 0..M-1
//   z = IDFT_M(Z) (unnormalised; the 1/N is already in K3)  =>  Phi_{2m} = Re z_m, Phi_{2m+1} = Im z_m.
// MODE 0: psi <- exp(-dt H) s1 psi                         (imaginary time, BJ:north_star (b))
// MODE 1: psi <- (cos(dt H) - i sin(dt H)) psi             (real time)
// MODE 2: no update; accumulates sum V n, sum n^2, sum Phi n, sum n     (observables, R#16)
// MODE 3: no update; writes Phi to phi_out (dgpe_dipolar)
//   H = V + g n + gdd Phi,  n = s2 |psi|^2,  V = 0.5 (vx[i] + vy[j] + vz[k]) with
//   vx[i] = gamma^2 x_i^2 etc. (P:L31 harmonic anisotropic trap; R#1, R#6).
// ------------------------------------------------------------------------------------------------
struct NonlinArgs {
    int nlines, ny, nz;
    double dt, g, gdd;
    const double *vx, *vy, *vz;
    const double* scal;
    double* partials;          // MODE 2
    unsigned int* ticket;      // MODE 2
    double* out;               // MODE 2: 4 totals;  MODE 3: phi_out
};

// DT = element type of psi: cplx, or double for the observables (MODE 2) of a real-valued psi (DGPE_IMAG_RPSI)
template <int MODE, typename DT>
__global__ void __launch_bounds__(512, 1) k_c2r_nonlin(DT* __restrict__ psi, const cplx* __restrict__ spec, FftPlan P,
                             const cplx* __restrict__ tws, NonlinArgs A)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cplx* sm = reinterpret_cast<cplx*>(smem_raw);
    __shared__ double red[32 * 4];
    const int c = threadIdx.x & 7, b = threadIdx.x >> 3, nb = blockDim.x >> 3;
    const int line = blockIdx.x * TILE_COLS + c;
    const bool valid = line < A.nlines;
    const int nz = A.nz, M = nz >> 1, nzh = M + 1;

    if (valid) {
        const cplx* in = spec + (long long)line * nzh;
        for (int k = b; k <= M; k += nb) sm[k * TILE_COLS + c] = in[k];
    }
    __syncthreads();
    if (valid) {
        for (int k = b; 2 * k <= M; k += nb) {
            const int k2 = M - k;
            cplx xa = sm[k * TILE_COLS + c], xb = sm[k2 * TILE_COLS + c];
            {
                cplx w = cconj(__ldg(&tws[k]));            // e^{+2 pi i k/nz}
                cplx s = cadd(xa, cconj(xb)), d = csub(xa, cconj(xb));
                cplx wd = cmul(w, d);
                sm[k * TILE_COLS + c] = mk(s.x - wd.y, s.y + wd.x);     // s + i wd
            }
            if (k2 != k && k2 < M) {
                cplx w = cconj(__ldg(&tws[k2]));
                cplx s = cadd(xb, cconj(xa)), d = csub(xb, cconj(xa));
                cplx wd = cmul(w, d);
                sm[k2 * TILE_COLS + c] = mk(s.x - wd.y, s.y + wd.x);
            }
        }
    }
    __syncthreads();

    fft_run<true>(P, b, valid && (b < P.nbf), sm + c, TILE_COLS, sm + c, TILE_COLS, sm + c, TILE_COLS);

    double acc[4] = {0.0, 0.0, 0.0, 0.0};
    if (valid) {
        const int i = line / A.ny, j = line - i * A.ny;
        const double vxy = __ldg(&A.vx[i]) + __ldg(&A.vy[j]);
        const double s2 = A.scal[SC_S2], s1 = A.scal[SC_S1];
        DT* p = psi + (long long)line * nz;
        for (int m = b; m < M; m += nb) {
            const cplx phi = sm[m * TILE_COLS + c];
            if (MODE == 3) {
                double* po = A.out + (long long)line * nz;
                po[2 * m] = phi.x;
                po[2 * m + 1] = phi.y;
                continue;
            }
            DT a[2] = {p[2 * m], p[2 * m + 1]};
            const double ph[2] = {phi.x, phi.y};
#pragma unroll
            for (int t = 0; t < 2; ++t) {
                const double dens = s2 * cabs2(a[t]);
                const double V = 0.5 * (vxy + __ldg(&A.vz[2 * m + t]));
                if constexpr (MODE == 2) {
                    acc[0] += V * dens;
                    acc[1] += dens * dens;
                    acc[2] += ph[t] * dens;
                    acc[3] += dens;
                } else if constexpr (sizeof(DT) == sizeof(cplx)) {
                    const double H = V + A.g * dens + A.gdd * ph[t];
                    if (MODE == 0) {
                        const double f = exp(-A.dt * H) * s1;
                        a[t] = mk(f * a[t].x, f * a[t].y);
                    } else {
                        double sn, cs;
                        sincos(A.dt * H, &sn, &cs);
                        a[t] = mk(cs * a[t].x + sn * a[t].y, cs * a[t].y - sn * a[t].x);
                    }
                }
            }
            if (MODE == 0 || MODE == 1) {
                p[2 * m] = a[0];
                p[2 * m + 1] = a[1];
            }
        }
    }
    if (MODE == 2) {
        double tot[4];
        if (grid_reduce<4>(acc, A.partials, A.ticket, tot, red)) {
#pragma unroll
            for (int t = 0; t < 4; ++t) A.out[t] = tot[t];
        }
    }
}

}  // namespace dgpe
