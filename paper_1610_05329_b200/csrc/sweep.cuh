// sweep.cuh -- Crank-Nicolson line sweeps K6/K7/K8 (BJ:north_star (c): "three ADI Crank-Nicolson
// sweeps along x, y and z, each a constant-coefficient tridiagonal forward/backward recursion per
// grid line with Dirichlet boundaries"), plus the folded norm reduction (BJ:north_star (d)).
//
// Per line p_0..p_{n-1} (end nodes are the Dirichlet boundary, read as 0 and written as 0; R#7, R#8):
//   d_j = r p_{j-1} + (1-2r) p_j + r p_{j+1}                     j = 1..n-2
//   e_j = (d_j + r e_{j-1}) inv_j,  e_0 = 0                      forward elimination
//   x_j = e_j - c_j x_{j+1},        x_{n-1} = 0                  back substitution
// with r = dt/(4 d^2) (imaginary time) or i dt/(4 d^2) (real time), and the elimination factors of
// the constant matrix tridiag(-r, 1+2r, -r):  inv_1 = 1/(1+2r), c_j = -r inv_j,
// inv_j = 1/((1+2r) + r c_{j-1})  (R#9) -- per-axis tables, not per-line data.
//
// Both recursions are first-order linear, so they are evaluated in chunks of Lc unknowns, one thread
// per (line, chunk), with the line tile resident in shared memory:
//   A  local forward recursion with zero inflow -> e'_j, chunk outflow E_g
//   B  inflow of chunk g:  ein_g = E_{g-1} + A_{g-1} (E_{g-2} + A_{g-2} (...)),  A_g = prod_{chunk} r inv_j;
//      the look-back stops after Kf chunks, where |A|^Kf < 2^-80 (decided on the host from the actual
//      tables: Kf = 2 for every BASELINE config, the full chain when r is large)
//   C  e_j = e'_j + F_j ein_g (F = running product of r inv_j inside the chunk), local backward
//      recursion with zero inflow -> x'_j, chunk outflow X_g
//   D  inflow from the right, same look-back with B_g = prod_{chunk} (-c_j), depth Kb
//   E  x_j = x'_j + G_j xin_g  (G = running product of -c_j from the chunk's right end)
// This is the exact solution of the tridiagonal system up to rounding (terms below 2^-80 of the
// line's largest entry are dropped); DESIGN.md section 6 has the derivation.
//
// Thread layout as in fft.cuh: c = tid & 7 is the line inside the tile, g = tid >> 3 the chunk, so a
// quarter-warp touches the 8 lines of one tile row: 128 contiguous bytes, no bank conflicts.  The tile
// row pitch is 9 for the z axis (lines are contiguous in global memory there, and the staging copy
// walks along a line: pitch 9 makes both access directions conflict free) and 8 for x and y.
#pragma once
#include "common.cuh"

namespace dgpe {

template <typename CT>
struct SweepTables {
    CT r;              // off-diagonal of B
    CT omr2;           // 1 - 2r
    const CT* inv;     // [n]   inv_j
    const CT* cc;      // [n]   c_j
    const CT* F;       // [n]   forward running product inside the chunk
    const CT* Gm;      // [n]   backward running product inside the chunk
    const CT* Ach;     // [G]   chunk forward factor
    const CT* Bch;     // [G]   chunk backward factor
    const CT* ztab;    // [8 Lc] compact table for CONSTTAB kernels: [inv, c, F, G] of chunk 0, then of the converged chunk
    int Lc, G, Kf, Kb;
    int gU;            // chunks gU .. G-2 have bit-identical table entries (G if none): a lane-per-chunk kernel
                       // may read chunk gU's entries for all of them (one broadcast address)
};

// The Thomas tables as kernel parameters (constant bank: operands of the fp64 instructions, no load
// instruction at all), valid when the elimination factors have converged to their fixed point by the
// second chunk -- decided on the host by a bitwise comparison of the table entries (AxisSweep::consttab).
// Chunk 0 uses its own entries, every other chunk the converged ones.  The forward inflow of chunk 0
// and the backward inflow of the last chunk are zero, so F of chunk 0 and Gm of the (possibly shorter)
// last chunk never matter.  Kernels take CONSTTAB = false to read the global tables instead (any r).
template <typename CT, int LC>
struct ChunkTabs {
    CT inv0[LC], cc0[LC], gm0[LC];
    CT invU[LC], ccU[LC], fU[LC], gmU[LC];
};

struct SweepFold {
    int enabled;              // accumulate sum |psi'|^2 and finish the norm in the last block
    double dV;
    double* partials;
    unsigned int* ticket;
    double* scal;
};

template <typename CT, bool ZAXIS>
__global__ void __launch_bounds__(512) k_sweep(cplx* __restrict__ psi, LineMap map, SweepTables<CT> T, SweepFold fold)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ double red[32];
    constexpr int PITCH = ZAXIS ? 9 : 8;
    const int n = map.n;
    cplx* sm = reinterpret_cast<cplx*>(smem_raw);          // [n][PITCH]
    cplx* smE = sm + (size_t)n * PITCH;                     // [G][8]
    cplx* smX = smE + (size_t)T.G * TILE_COLS;              // [G][8]
    const int tid = threadIdx.x, nthr = blockDim.x;
    const int col0 = blockIdx.x * TILE_COLS;
    cplx* base = psi + (long long)blockIdx.y * map.batch_stride;

    // ---- stage the tile (faces read as zero) ----
    if (ZAXIS) {
        for (int t = tid; t < n * TILE_COLS; t += nthr) {
            const int l = t / n, j = t - l * n;
            const int col = col0 + l;
            cplx v = mk(0.0, 0.0);
            if (col < map.ncols && j > 0 && j < n - 1)
                v = base[(long long)col * map.col_stride + (long long)j * map.elem_stride];
            sm[j * PITCH + l] = v;
        }
    } else {
        for (int t = tid; t < n * TILE_COLS; t += nthr) {
            const int j = t >> 3, l = t & 7;
            const int col = col0 + l;
            cplx v = mk(0.0, 0.0);
            if (col < map.ncols && j > 0 && j < n - 1)
                v = base[(long long)col * map.col_stride + (long long)j * map.elem_stride];
            sm[j * PITCH + l] = v;
        }
    }
    __syncthreads();

    const int c = tid & 7, g = tid >> 3;
    const bool work = g < T.G;
    const int s = 1 + g * T.Lc;
    const int t_end = min(s + T.Lc, n - 1);
    cplx* col_sm = sm + c;

    // neighbours across the chunk borders, before anything is overwritten
    cplx pm = mk(0.0, 0.0), pt = mk(0.0, 0.0);
    if (work) {
        pm = col_sm[(s - 1) * PITCH];
        pt = col_sm[t_end * PITCH];
    }
    __syncthreads();

    // ---- A: local forward ----
    if (work) {
        cplx e = mk(0.0, 0.0);
        cplx p0 = col_sm[s * PITCH];
        for (int j = s; j < t_end; ++j) {
            const cplx pp = (j + 1 < t_end) ? col_sm[(j + 1) * PITCH] : pt;
            cplx d = coef_mul(T.r, cadd(pm, pp));
            d = coef_fma(T.omr2, p0, d);
            d = coef_fma(T.r, e, d);
            e = coef_mul(__ldg(&T.inv[j]), d);
            col_sm[j * PITCH] = e;
            pm = p0;
            p0 = pp;
        }
        smE[g * TILE_COLS + c] = e;
    }
    __syncthreads();

    // ---- B + C: forward inflow, local backward ----
    if (work) {
        cplx ein = mk(0.0, 0.0);
        for (int h = max(0, g - T.Kf); h < g; ++h) ein = coef_fma(__ldg(&T.Ach[h]), ein, smE[h * TILE_COLS + c]);
        cplx x = mk(0.0, 0.0);
        for (int j = t_end - 1; j >= s; --j) {
            cplx e = coef_fma(__ldg(&T.F[j]), ein, col_sm[j * PITCH]);
            // x = e - c_j x
            CT cj = __ldg(&T.cc[j]);
            cplx cx = coef_mul(cj, x);
            x = csub(e, cx);
            col_sm[j * PITCH] = x;
        }
        smX[g * TILE_COLS + c] = x;
    }
    __syncthreads();

    // ---- D + E: backward inflow, final values ----
    if (work) {
        cplx xin = mk(0.0, 0.0);
        for (int h = min(T.G - 1, g + T.Kb); h > g; --h) xin = coef_fma(__ldg(&T.Bch[h]), xin, smX[h * TILE_COLS + c]);
        for (int j = s; j < t_end; ++j) col_sm[j * PITCH] = coef_fma(__ldg(&T.Gm[j]), xin, col_sm[j * PITCH]);
    }
    __syncthreads();

    // ---- write back (rows 0 and n-1 of the tile are still zero: the Dirichlet faces) ----
    double nrm = 0.0;
    if (ZAXIS) {
        for (int t = tid; t < n * TILE_COLS; t += nthr) {
            const int l = t / n, j = t - l * n;
            const int col = col0 + l;
            if (col < map.ncols) {
                cplx v = sm[j * PITCH + l];
                nrm += cabs2(v);
                base[(long long)col * map.col_stride + (long long)j * map.elem_stride] = v;
            }
        }
    } else {
        for (int t = tid; t < n * TILE_COLS; t += nthr) {
            const int j = t >> 3, l = t & 7;
            const int col = col0 + l;
            if (col < map.ncols) {
                cplx v = sm[j * PITCH + l];
                nrm += cabs2(v);
                base[(long long)col * map.col_stride + (long long)j * map.elem_stride] = v;
            }
        }
    }

    if (fold.enabled) {
        double v[1] = {nrm}, tot[1];
        if (grid_reduce<1>(v, fold.partials, fold.ticket, tot, red)) {
            const double norm = tot[0] * fold.dV;
            fold.scal[SC_NORM] = norm;
            fold.scal[SC_S2] = 1.0 / norm;
            fold.scal[SC_S1] = 1.0 / sqrt(norm);
            if (!(norm > 0.0) || !isfinite(norm)) fold.scal[SC_BAD] = 1.0;
        }
    }
}

// psi <- psi * scal[SC_S1]   (the explicit renormalisation at the end of dgpe_step)
__global__ void k_scale(cplx* __restrict__ psi, long long N, const double* __restrict__ scal)
{
    const double s = scal[SC_S1];
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long p = blockIdx.x * (long long)blockDim.x + threadIdx.x; p < N; p += stride) {
        cplx v = psi[p];
        psi[p] = mk(v.x * s, v.y * s);
    }
}

__global__ void k_set_scal(double* scal, double s2, double s1, int clear_bad)
{
    scal[SC_S2] = s2;
    scal[SC_S1] = s1;
    if (clear_bad) scal[SC_BAD] = 0.0;
}

// scal <- the scale factors of a norm that was summed over the ranks of a slab decomposition (dgpe_slab): the
// folded reduction of the last sweep only knows its own slab's part
__global__ void k_set_norm(double* scal, const double* __restrict__ norm_total)
{
    const double norm = *norm_total;
    scal[SC_NORM] = norm;
    scal[SC_S2] = 1.0 / norm;
    scal[SC_S1] = 1.0 / sqrt(norm);
    if (!(norm > 0.0) || !isfinite(norm)) scal[SC_BAD] = 1.0;
}

}  // namespace dgpe
