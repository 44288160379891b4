// xysweep.cuh -- K6 / K7: the Crank-Nicolson sweeps along the strided axes x and y with every chunk of
// a line held in registers (SV section 8a rows a6, a7; BJ:north_star (c) "constant-coefficient
// tridiagonal forward/backward recursion per grid line with Dirichlet boundaries", and "for the x and y
// sweeps, adjacent threads own adjacent z-lines, so loads coalesce naturally").
//
// Algorithm and tables as k_sweep (sweep.cuh): both recursions of the Thomas solve are first-order
// linear with tabulated constant coefficients, so a line is cut into chunks of LC unknowns, one thread
// per (line, chunk), and the chunks are coupled by a short look-back over the chunk outflows.
// Here thread (c = tid & 7, g = tid >> 3) loads its LC (+2 neighbour) values of line c straight from
// global memory (a quarter-warp reads the 8 lines of one row: 128 contiguous bytes), runs the local
// forward and backward recursions in registers, and stores the final values straight back; only the
// two chunk outflows per thread (E_g, X_g) pass through shared memory.  psi moves once in and once
// out: 32N bytes per sweep.
//
// With `fold.enabled` the kernel also accumulates sum |psi'|^2 and the last block finishes the norm
// (BJ:north_star (d): "norm ... warp-shuffle plus block reductions, with the rescale folded into the
// next kernel").
#pragma once
#include "ctfft.cuh"
#include "sweep.cuh"

namespace dgpe {

// grid = (ceil(ncols/8), nbatch); block = 8*G rounded up to a warp multiple (<= NTMAX)
// pf_tiles > 0: every CTA asks L2 for the tile that will be processed pf_tiles CTAs later.
template <typename CT, int LC, bool CONSTTAB, int NTMAX, int MINB>
__global__ void __launch_bounds__(NTMAX, MINB)
k_sweep_xy(cplx* __restrict__ psi, LineMap map, SweepTables<CT> T, SweepFold fold, int pf_tiles,
           const __grid_constant__ ChunkTabs<CT, LC> P)
{
    __shared__ cplx smE[NTMAX / 8][TILE_COLS];
    __shared__ cplx smX[NTMAX / 8][TILE_COLS];
    __shared__ double red[32];
    const int n = map.n;
    const int tid = threadIdx.x, c = tid & 7, g = tid >> 3;
    const int col = blockIdx.x * TILE_COLS + c;
    const bool colok = col < map.ncols;
    const bool work = colok && g < T.G;
    const int s = 1 + g * LC;
    const int t_end = min(s + LC, n - 1);
    const int cnt = t_end - s;                     // unknowns of this chunk (<= 0 for idle threads)
    cplx* gp = psi + (long long)blockIdx.y * map.batch_stride + (long long)(colok ? col : 0) * map.col_stride;
    const long long es = map.elem_stride;

    if (pf_tiles > 0) {
        const long long id = (long long)blockIdx.y * gridDim.x + blockIdx.x + pf_tiles;
        const int by = (int)(id / gridDim.x), bx = (int)(id - (long long)by * gridDim.x);
        if (by < (int)gridDim.y)
            for (int j = tid; j < n; j += blockDim.x)
                prefetch_l2(psi + (long long)by * map.batch_stride + (long long)bx * TILE_COLS * map.col_stride + (long long)j * es);
    }
    const bool g0 = g == 0;
    // (kernel parameters here: read through L1 instead, as the TMA sweep and the z kernels do, this kernel -- whose loads
    // already wait on memory -- got slower: 512^3 x sweep 0.82 -> 1.09 ms)
    auto t_inv = [&](int i) { if constexpr (CONSTTAB) return g0 ? P.inv0[i] : P.invU[i]; else return __ldg(&T.inv[s + i]); };
    auto t_cc = [&](int i) { if constexpr (CONSTTAB) return g0 ? P.cc0[i] : P.ccU[i]; else return __ldg(&T.cc[s + i]); };
    auto t_F = [&](int i) { if constexpr (CONSTTAB) return P.fU[i]; else return __ldg(&T.F[s + i]); };
    auto t_Gm = [&](int i) { if constexpr (CONSTTAB) return g0 ? P.gm0[i] : P.gmU[i]; else return __ldg(&T.Gm[s + i]); };

    // ---- load p_{s-1} .. p_{t_end}; the end nodes of the line are read as zero (R#7, R#8) ----
    cplx p[LC + 2];
#pragma unroll
    for (int i = 0; i < LC + 2; ++i) {
        const int j = s - 1 + i;
        p[i] = mk(0.0, 0.0);
        if (work && j >= 1 && j <= n - 2 && i <= cnt + 1) p[i] = ld_stream(gp + (long long)j * es);
    }

    // ---- A: local forward elimination with zero inflow ----
    cplx ev[LC];
    cplx e = mk(0.0, 0.0);
#pragma unroll
    for (int i = 0; i < LC; ++i) {
        ev[i] = mk(0.0, 0.0);
        if (work && i < cnt) {
            // e_j = inv_j (d_j + r e_{j-1}) written as inv_j d_j + (r inv_j) e_{j-1}, r inv_j = -c_j: one
            // dependent fma per unknown instead of an fma and a multiply
            const cplx d = cn_rhs(T.r, T.omr2, p[i], p[i + 1], p[i + 2]);
            e = coef_fma(coef_neg(t_cc(i)), e, coef_mul(t_inv(i), d));
            ev[i] = e;
        }
    }
    if (g < T.G) smE[g][c] = e;
    __syncthreads();

    // ---- B + C: forward inflow, local back substitution with zero inflow ----
    cplx x = mk(0.0, 0.0);
    if (work) {
        cplx ein = mk(0.0, 0.0);
        for (int h = max(0, g - T.Kf); h < g; ++h) ein = coef_fma(__ldg(&T.Ach[h]), ein, smE[h][c]);
#pragma unroll
        for (int i = LC - 1; i >= 0; --i) {
            if (i < cnt) {
                const cplx ee = coef_fma(t_F(i), ein, ev[i]);
                x = coef_fma(coef_neg(t_cc(i)), x, ee);
                ev[i] = x;
            }
        }
    }
    if (g < T.G) smX[g][c] = x;
    __syncthreads();

    // ---- D + E: backward inflow, final values straight to global memory ----
    double nrm = 0.0;
    if (work) {
        cplx xin = mk(0.0, 0.0);
        for (int h = min(T.G - 1, g + T.Kb); h > g; --h) xin = coef_fma(__ldg(&T.Bch[h]), xin, smX[h][c]);
        if (g == 0) st_stream(gp, mk(0.0, 0.0));
        if (t_end == n - 1) st_stream(gp + (long long)(n - 1) * es, mk(0.0, 0.0));
#pragma unroll
        for (int i = 0; i < LC; ++i) {
            if (i < cnt) {
                const cplx v = coef_fma(t_Gm(i), xin, ev[i]);
                nrm += cabs2(v);
                st_stream(gp + (long long)(s + i) * es, v);
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

}  // namespace dgpe
