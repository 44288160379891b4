// observe.cuh -- reductions behind dgpe_norm / dgpe_rms / dgpe_chempot / dgpe_energy (R#14-R#17).
// Not on the timed path: plain coalesced grid-stride kernels with the deterministic grid_reduce.
#pragma once
#include "common.cuh"

namespace dgpe {

struct ObsArgs {
    int nx, ny, nz;
    const double *x2, *y2, *z2;    // squared coordinates x_i^2 = ((i - n/2) d)^2   (R#6)
    double* partials;
    unsigned int* ticket;
    double* out;
};

// out[0..3] = sum n, sum x^2 n, sum y^2 n, sum z^2 n      (n = |psi|^2)
// DT = cplx, or double for a real-valued psi (DGPE_IMAG_RPSI)
template <typename DT>
__global__ void k_moments(const DT* __restrict__ psi, ObsArgs A)
{
    __shared__ double red[32 * 4];
    double acc[4] = {0.0, 0.0, 0.0, 0.0};
    const int nlines = A.nx * A.ny;
    for (int line = blockIdx.x; line < nlines; line += gridDim.x) {
        const int i = line / A.ny, j = line - i * A.ny;
        const double xx = __ldg(&A.x2[i]), yy = __ldg(&A.y2[j]);
        const DT* p = psi + (long long)line * A.nz;
        for (int k = threadIdx.x; k < A.nz; k += blockDim.x) {
            const double n = cabs2(p[k]);
            acc[0] += n;
            acc[1] += xx * n;
            acc[2] += yy * n;
            acc[3] += __ldg(&A.z2[k]) * n;
        }
    }
    double tot[4];
    if (grid_reduce<4>(acc, A.partials, A.ticket, tot, red)) {
#pragma unroll
        for (int t = 0; t < 4; ++t) A.out[t] = tot[t];
    }
}

// out[0..2] = sum over links along x, y, z of |psi_{j+1} - psi_j|^2, links j = -1..n-1 with the
// ghost nodes psi_{-1} = psi_n = 0   (R#16)
template <typename DT>
__global__ void k_kinetic(const DT* __restrict__ psi, ObsArgs A)
{
    __shared__ double red[32 * 3];
    double acc[3] = {0.0, 0.0, 0.0};
    const int nlines = A.nx * A.ny;
    const long long sy = A.nz, sx = (long long)A.ny * A.nz;
    for (int line = blockIdx.x; line < nlines; line += gridDim.x) {
        const int i = line / A.ny, j = line - i * A.ny;
        const DT* p = psi + (long long)line * A.nz;
        for (int k = threadIdx.x; k < A.nz; k += blockDim.x) {
            const DT here = p[k];
            const DT zero = DT();
            const DT px = (i + 1 < A.nx) ? p[k + sx] : zero;
            const DT py = (j + 1 < A.ny) ? p[k + sy] : zero;
            const DT pz = (k + 1 < A.nz) ? p[k + 1] : zero;
            acc[0] += cabs2(csub(px, here));
            acc[1] += cabs2(csub(py, here));
            acc[2] += cabs2(csub(pz, here));
            if (i == 0) acc[0] += cabs2(here);
            if (j == 0) acc[1] += cabs2(here);
            if (k == 0) acc[2] += cabs2(here);
        }
    }
    double tot[3];
    if (grid_reduce<3>(acc, A.partials, A.ticket, tot, red)) {
#pragma unroll
        for (int t = 0; t < 3; ++t) A.out[t] = tot[t];
    }
}

}  // namespace dgpe
