// xysweep_tma.cuh -- K6 / K7 as a persistent, TMA-fed pipeline (SV section 8a rows a6, a7, a9).
//
// Same algorithm as k_sweep_xy (xysweep.cuh: one thread per (line, chunk of 8 unknowns), recursions in
// registers, chunk outflows through shared memory); what changes is how the tile moves.  One CTA per SM
// walks the tiles blockIdx.x, blockIdx.x + gridDim.x, ...; a tile (8 lines x the whole line, [n][8]
// complex = n rows of 128 bytes) is fetched by the Tensor Memory Accelerator (cp.async.bulk.tensor, boxes
// of up to 256 rows, completion on an mbarrier) into one of NSTAGE shared-memory stages while the CTA
// computes on another, and the results go back through the same stage by a TMA tensor store.  No
// thread issues a global load or store: HBM latency is covered by the depth of the pipeline (one to two
// tiles in flight per SM), not by occupancy, so the kernel is as good at n = 768 (96 KB tiles, one CTA
// of 768 threads per SM) as at n = 512.
//
// The tensor map (host: dgpe_api.cu) is rank 3 over psi viewed as doubles: x sweep {2 ny nz, nx, 1},
// y sweep {2 nz, ny, nx}; a tile is the box {16 doubles, rows, 1}.
#pragma once
#include "tma.cuh"
#include "xysweep.cuh"
#include <type_traits>

namespace dgpe {

struct TmaWalk {
    int n;                 // line length (rows of a tile)
    int box_rows;          // rows per TMA box (<= 256, divides n)
    int tiles_per_batch;   // ncols / 8
    int ntiles;            // tiles_per_batch * nbatch
};

constexpr int TMA_LC = 8;

// grid = min(ntiles, #SMs * resident CTAs); block = 8*G rounded to a warp multiple (<= NTMAX);
// dynamic smem = NSTAGE * n * 128 bytes (+128 for alignment)
template <typename CT, bool CONSTTAB, int NSTAGE, int NTMAX>
__global__ void __launch_bounds__(NTMAX, 1)
k_sweep_tma(const __grid_constant__ CUtensorMap tmap, TmaWalk W, SweepTables<CT> T, SweepFold fold,
            const __grid_constant__ ChunkTabs<CT, TMA_LC> P)
{
    constexpr int LC = TMA_LC;
    extern __shared__ unsigned char smem_dyn[];
    __shared__ cplx smE[NTMAX / 8][TILE_COLS];
    __shared__ cplx smX[NTMAX / 8][TILE_COLS];
    __shared__ double red[32];
    __shared__ __align__(8) unsigned long long full[NSTAGE];
    // 128-byte aligned start of the stages, as an OFFSET into the shared array: the pointer keeps its address space, so
    // the tile accesses compile to LDS/STS (through a round trip over an integer they were generic LD.E/ST.E)
    cplx* stages = reinterpret_cast<cplx*>(smem_dyn + ((128u - (smem_addr(smem_dyn) & 127u)) & 127u));
    const int n = W.n;
    const int tile_elems = n * TILE_COLS;
    const unsigned tile_bytes = (unsigned)tile_elems * 16u;
    const int tid = threadIdx.x, c = tid & 7, g = tid >> 3;
    const bool work = g < T.G;
    const int s = 1 + g * LC;
    const int t_end = min(s + LC, n - 1);
    const int cnt = t_end - s;
    const int first = blockIdx.x, stride = gridDim.x;
    const int nmine = (first < W.ntiles) ? (W.ntiles - first + stride - 1) / stride : 0;

    // Table entries.  With CONSTTAB only chunk 0 differs from the converged entries, and chunk 0 lives in warp 0:
    // the other warps take the MIXED = false instantiation of each phase, whose table operands are plain
    // constant-bank reads with no per-element select.
    // (It pays with complex tables, real time: 768-point y sweep 1.64 -> 1.24 ms; with real tables the plain
    // selects are as fast, so there every warp takes the MIXED path.)
    const bool g0 = g == 0;
    using MixedT = std::true_type;
    using PlainT = std::false_type;
    // Real tables (imaginary time): ONE compact table read through L1, the chunk-0 / converged-chunk choice in the address
    // (T.ztab; as kernel parameters every selected double costs three LDC and the constant-load unit was 43 % busy):
    // 512^3 y sweep 0.774 -> 0.686 ms (0.955 of measured peak), real-valued psi 0.39 -> 0.35 ms.  Complex tables (real
    // time) keep the parameters with the per-warp split below (768-point sweeps: 1.23 vs 1.28 ms).
    constexpr bool LDGTAB = CONSTTAB && sizeof(CT) == sizeof(double);
    constexpr bool SPLIT = CONSTTAB && !LDGTAB;
    const bool warp0 = tid < 32;
    auto run = [&](auto&& phase) {
        if constexpr (SPLIT) { if (warp0) phase(MixedT{}); else phase(PlainT{}); }
        else phase(MixedT{});
    };
    const CT* tb = T.ztab + (g0 ? 0 : 4 * LC);
    auto t_inv = [&](auto M, int i) {
        if constexpr (!CONSTTAB) return __ldg(&T.inv[s + i]);
        else if constexpr (LDGTAB) return __ldg(&tb[i]);
        else if constexpr (decltype(M)::value) return g0 ? P.inv0[i] : P.invU[i];
        else return P.invU[i];
    };
    auto t_cc = [&](auto M, int i) {
        if constexpr (!CONSTTAB) return __ldg(&T.cc[s + i]);
        else if constexpr (LDGTAB) return __ldg(&tb[LC + i]);
        else if constexpr (decltype(M)::value) return g0 ? P.cc0[i] : P.ccU[i];
        else return P.ccU[i];
    };
    auto t_F = [&](auto M, int i) {
        if constexpr (!CONSTTAB) return __ldg(&T.F[s + i]);
        else if constexpr (LDGTAB) return __ldg(&tb[2 * LC + i]);
        else return P.fU[i];
    };
    auto t_Gm = [&](auto M, int i) {
        if constexpr (!CONSTTAB) return __ldg(&T.Gm[s + i]);
        else if constexpr (LDGTAB) return __ldg(&tb[3 * LC + i]);
        else if constexpr (decltype(M)::value) return g0 ? P.gm0[i] : P.gmU[i];
        else return P.gmU[i];
    };

    auto coords = [&](int it, int& c0, int& c2) {
        const int t = first + it * stride;
        const int bat = t / W.tiles_per_batch;
        c0 = (t - bat * W.tiles_per_batch) * (2 * TILE_COLS);
        c2 = bat;
    };
    auto issue_load = [&](int it) {                     // thread 0 only
        int c0, c2;
        coords(it, c0, c2);
        const int st = it % NSTAGE;
        mbar_expect_tx(&full[st], tile_bytes);
        for (int r0 = 0; r0 < n; r0 += W.box_rows)
            tma_load_3d(stages + (size_t)st * tile_elems + (size_t)r0 * TILE_COLS, &tmap, c0, r0, c2, &full[st]);
    };

    if (tid == 0) {
        for (int st = 0; st < NSTAGE; ++st) mbar_init(&full[st], 1);
        mbar_fence_init();
    }
    __syncthreads();
    if (tid == 0)
        for (int it = 0; it < NSTAGE - 1 && it < nmine; ++it) issue_load(it);

    double nrm = 0.0;
    for (int it = 0; it < nmine; ++it) {
        const int st = it % NSTAGE;
        cplx* tile = stages + (size_t)st * tile_elems;
        cplx* col = tile + c;
        mbar_wait(&full[st], (unsigned)((it / NSTAGE) & 1));

        // ---- p_{s-1} .. p_{t_end} from the tile; the end nodes of the line are read as zero (R#7, R#8) ----
        cplx p[LC + 2];
#pragma unroll
        for (int i = 0; i < LC + 2; ++i) {
            const int j = s - 1 + i;
            p[i] = mk(0.0, 0.0);
            if (work && j >= 1 && j <= n - 2 && i <= cnt + 1) p[i] = col[j * TILE_COLS];
        }
        // ---- A: local forward elimination with zero inflow ----
        cplx ev[LC];
        cplx e = mk(0.0, 0.0);
        auto phaseA = [&](auto M) {
#pragma unroll
            for (int i = 0; i < LC; ++i) {
                ev[i] = mk(0.0, 0.0);
                if (work && i < cnt) {
                    const cplx d = cn_rhs(T.r, T.omr2, p[i], p[i + 1], p[i + 2]);
                    e = coef_fma(coef_neg(t_cc(M, i)), e, coef_mul(t_inv(M, i), d));
                    ev[i] = e;
                }
            }
        };
        run(phaseA);
        if (work) smE[g][c] = e;
        __syncthreads();                                 // every thread has read its part of the tile

        // the stage tile it-1 used is free once its store has read shared memory: refill it now, one
        // compute phase after that store was issued
        if (tid == 0 && it + NSTAGE - 1 < nmine) {
            tma_store_wait_read<0>();
            issue_load(it + NSTAGE - 1);
        }

        // ---- B + C: forward inflow, local back substitution with zero inflow ----
        cplx x = mk(0.0, 0.0);
        if (work) {
            cplx ein = mk(0.0, 0.0);
            for (int h = max(0, g - T.Kf); h < g; ++h) ein = coef_fma(__ldg(&T.Ach[h]), ein, smE[h][c]);
            auto phaseC = [&](auto M) {
#pragma unroll
                for (int i = LC - 1; i >= 0; --i) {
                    if (i < cnt) {
                        const cplx ee = coef_fma(t_F(M, i), ein, ev[i]);
                        x = coef_fma(coef_neg(t_cc(M, i)), x, ee);
                        ev[i] = x;
                    }
                }
            };
            run(phaseC);
            smX[g][c] = x;
        }
        __syncthreads();

        // ---- D + E: backward inflow, final values back into the tile ----
        if (work) {
            cplx xin = mk(0.0, 0.0);
            for (int h = min(T.G - 1, g + T.Kb); h > g; --h) xin = coef_fma(__ldg(&T.Bch[h]), xin, smX[h][c]);
            if (g == 0) col[0] = mk(0.0, 0.0);
            if (t_end == n - 1) col[(n - 1) * TILE_COLS] = mk(0.0, 0.0);
            auto phaseE = [&](auto M) {
#pragma unroll
                for (int i = 0; i < LC; ++i) {
                    if (i < cnt) {
                        const cplx v = coef_fma(t_Gm(M, i), xin, ev[i]);
                        nrm += cabs2(v);
                        col[(s + i) * TILE_COLS] = v;
                    }
                }
            };
            run(phaseE);
        }
        fence_proxy_async();                             // my tile writes -> visible to the TMA store
        __syncthreads();
        if (tid == 0) {
            int c0, c2;
            coords(it, c0, c2);
            for (int r0 = 0; r0 < n; r0 += W.box_rows) tma_store_3d(&tmap, c0, r0, c2, tile + (size_t)r0 * TILE_COLS);
            tma_store_commit();
        }
    }
    if (tid == 0) tma_store_wait<0>();

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
