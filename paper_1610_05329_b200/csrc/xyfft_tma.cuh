// xyfft_tma.cuh -- K2 / K4 (FFT of the half-spectrum along y) as a persistent, TMA-fed pipeline.
//
// Same passes as k_fft_xy (xyfft.cuh, ctfft.cuh); what changes is how the tile moves, exactly as in
// xysweep_tma.cuh: one CTA per SM walks the tiles, the Tensor Memory Accelerator fetches tile i+1 (and
// i+2) into another shared-memory stage while the CTA transforms tile i in place, and the result leaves
// by a TMA tensor store from the same stage.  The rows of a tile start at multiples of 16 bytes only
// (nz/2+1 is odd), which the TMA does not mind, and the ragged last tile of a row (one valid kz bin out
// of 8 at nz/2+1 = 257) is zero-filled on load and clipped on store by the tensor map bounds.
//
// Tensor map (host): rank 3 over the half-spectrum viewed as doubles, {2 (nz/2+1), ny, nx}; a tile is
// the box {16 doubles, rows, 1}.
#pragma once
#include "xyfft.cuh"
#include "xysweep_tma.cuh"

namespace dgpe {

// grid = min(ntiles, #SMs); block = xy_threads<N>(); dynamic smem = NSTAGE * N * 128 bytes (+128)
template <int N, bool INV, int NSTAGE>
__global__ void __launch_bounds__(xy_threads<N>(), 1)
k_fft_tma(const __grid_constant__ CUtensorMap tmap, TmaWalk W, const cplx* __restrict__ tw)
{
    constexpr int NBF = xy_nbf<N>();
    constexpr int L = ct::npass(N);
    static_assert(L >= 2, "the pipelined kernel is for the long lines");
    extern __shared__ unsigned char smem_dyn[];
    __shared__ __align__(8) unsigned long long full[NSTAGE];
    // 128-byte aligned start of the stages, as an OFFSET into the shared array: the pointer keeps its address space, so
    // the tile accesses compile to LDS/STS (through a round trip over an integer they were generic LD.E/ST.E)
    cplx* stages = reinterpret_cast<cplx*>(smem_dyn + ((128u - (smem_addr(smem_dyn) & 127u)) & 127u));
    constexpr int tile_elems = N * TILE_COLS;
    constexpr unsigned tile_bytes = (unsigned)tile_elems * 16u;
    const int tid = threadIdx.x, c = tid & 7, b = tid >> 3;
    const bool on = b < NBF;
    const int first = blockIdx.x, stride = gridDim.x;
    const int nmine = (first < W.ntiles) ? (W.ntiles - first + stride - 1) / stride : 0;

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
        for (int r0 = 0; r0 < N; r0 += W.box_rows)
            tma_load_3d(stages + (size_t)st * tile_elems + (size_t)r0 * TILE_COLS, &tmap, c0, r0, c2, &full[st]);
    };

    if (tid == 0) {
        for (int st = 0; st < NSTAGE; ++st) mbar_init(&full[st], 1);
        mbar_fence_init();
    }
    __syncthreads();
    if (tid == 0)
        for (int it = 0; it < NSTAGE - 1 && it < nmine; ++it) issue_load(it);

    for (int it = 0; it < nmine; ++it) {
        const int st = it % NSTAGE;
        cplx* tile = stages + (size_t)st * tile_elems;
        cplx* col = tile + c;
        mbar_wait(&full[st], (unsigned)((it / NSTAGE) & 1));

        // pass 0 by hand, so that the refill of the stage tile it-1 used can be issued after its barrier
        CtPass<N, 0, INV, false, NBF> p0;
        if (on) p0.load(b, [&](int idx) { return col[PosTile::at(idx)]; });
        __syncthreads();                                 // every read of pass 0 precedes its writes
        if (tid == 0 && it + NSTAGE - 1 < nmine) {
            tma_store_wait_read<0>();                    // the store of tile it-1 has read its stage
            issue_load(it + NSTAGE - 1);
        }
        if (on) {
            p0.bfly(b);
            p0.scatter(b, [&](int idx, cplx val) { col[PosTile::at(idx)] = val; });
        }
        CtPass<N, 1, INV, false, NBF> p1;
        if (on) p1.load_tw(b, tw);                       // overlaps the barrier wait
        __syncthreads();
        auto none = [](int) { return mk(0.0, 0.0); };
        ct_fft_range_tw<N, INV, false, NBF, SyncCta, PosTile, 1, L, false>(
            p1, col, b, on, tw, none, [&](int idx, cplx val) { col[PosTile::at(idx)] = val; });

        fence_proxy_async();                             // my tile writes -> visible to the TMA store
        __syncthreads();
        if (tid == 0) {
            int c0, c2;
            coords(it, c0, c2);
            for (int r0 = 0; r0 < N; r0 += W.box_rows) tma_store_3d(&tmap, c0, r0, c2, tile + (size_t)r0 * TILE_COLS);
            tma_store_commit();
        }
    }
    if (tid == 0) tma_store_wait<0>();
}

// K3 (FFT along x, Udd~(k)/N, inverse FFT along x: xyfft.cuh FFT_X_UDD) on the same pipeline.  The tensor map is
// rank 3 over the half-spectrum viewed as doubles, {2 ny (nz/2+1), nx, 1}: a tile is 8 neighbouring flattened
// (ky, kz) columns x all nx rows, rows ny (nz/2+1) 16 bytes apart.
template <int N, int NSTAGE>
__global__ void __launch_bounds__(xy_threads<N>(), 1)
k_fft_tma_xudd(const __grid_constant__ CUtensorMap tmap, TmaWalk W, const cplx* __restrict__ tw, UddArgs U, int ncols)
{
    constexpr int NBF = xy_nbf<N>();
    constexpr int L = ct::npass(N);
    static_assert(L >= 2, "the pipelined kernel is for the long lines");
    extern __shared__ unsigned char smem_dyn[];
    __shared__ __align__(8) unsigned long long full[NSTAGE];
    // 128-byte aligned start of the stages, as an OFFSET into the shared array: the pointer keeps its address space, so
    // the tile accesses compile to LDS/STS (through a round trip over an integer they were generic LD.E/ST.E)
    cplx* stages = reinterpret_cast<cplx*>(smem_dyn + ((128u - (smem_addr(smem_dyn) & 127u)) & 127u));
    constexpr int tile_elems = N * TILE_COLS;
    constexpr unsigned tile_bytes = (unsigned)tile_elems * 16u;
    const int tid = threadIdx.x, c = tid & 7, b = tid >> 3;
    const bool on = b < NBF;
    const int first = blockIdx.x, stride = gridDim.x;
    const int nmine = (first < W.ntiles) ? (W.ntiles - first + stride - 1) / stride : 0;

    auto issue_load = [&](int it) {                     // thread 0 only
        const int st = it % NSTAGE;
        const int c0 = (first + it * stride) * (2 * TILE_COLS);
        mbar_expect_tx(&full[st], tile_bytes);
        for (int r0 = 0; r0 < N; r0 += W.box_rows)
            tma_load_3d(stages + (size_t)st * tile_elems + (size_t)r0 * TILE_COLS, &tmap, c0, r0, 0, &full[st]);
    };

    if (tid == 0) {
        for (int st = 0; st < NSTAGE; ++st) mbar_init(&full[st], 1);
        mbar_fence_init();
    }
    __syncthreads();
    if (tid == 0)
        for (int it = 0; it < NSTAGE - 1 && it < nmine; ++it) issue_load(it);

    auto none = [](int) { return mk(0.0, 0.0); };
    for (int it = 0; it < nmine; ++it) {
        const int st = it % NSTAGE;
        cplx* tile = stages + (size_t)st * tile_elems;
        cplx* col = tile + c;
        auto put = [&](int idx, cplx val) { col[PosTile::at(idx)] = val; };
        // ky^2, kz^2 of this thread's column (columns past the end of a ragged last tile: zero-filled by the
        // load, clipped by the store; they take the last column's wave numbers)
        const int cidx = min((first + it * stride) * TILE_COLS + c, ncols - 1);
        const int ky = cidx / U.nzh, kz = cidx - ky * U.nzh;
        const double qy = __ldg(&U.ky2[ky]), qz = __ldg(&U.kz2[kz]);
        mbar_wait(&full[st], (unsigned)((it / NSTAGE) & 1));

        // forward pass 0 by hand, so that the refill of the stage tile it-1 used can be issued after its barrier
        CtPass<N, 0, false, false, NBF> p0;
        if (on) { p0.load_tw(b, tw); p0.load(b, [&](int idx) { return col[PosTile::at(idx)]; }); }
        __syncthreads();
        if (tid == 0 && it + NSTAGE - 1 < nmine) {
            tma_store_wait_read<0>();
            issue_load(it + NSTAGE - 1);
        }
        if (on) {
            p0.bfly(b);
            p0.scatter(b, put);
        }
        if constexpr (L > 2) {
            CtPass<N, 1, false, false, NBF> p1;
            if (on) p1.load_tw(b, tw);
            __syncthreads();
            ct_fft_range_tw<N, false, false, NBF, SyncCta, PosTile, 1, L - 1, false>(p1, col, b, on, tw, none, put);
        } else {
            __syncthreads();
        }
        // last forward pass, Udd~(k)/N, first inverse pass: one set of registers (as k_fft_xy<N, FFT_X_UDD>)
        using PF = CtPass<N, L - 1, false, false, NBF>;
        using PI = CtPass<N, 0, true, true, NBF>;
        static_assert(PF::R == PI::R && PF::NB == PI::NB && PI::Ns == 1, "forward-last and inverse-first passes must match");
        PF pf;
        if (on) {
            pf.load_tw(b, tw);
            pf.load(b, [&](int idx) { return col[PosTile::at(idx)]; });
        }
        __syncthreads();
        PI pi;
        if (on) {
            pf.bfly(b);
            const double FOUR_PI_3 = 4.1887902047863909846168578443727;
            pf.modify(b, [&](int idx, cplx v) {
                const double kx = (double)(idx <= N / 2 ? idx : idx - N) * U.dkx;
                const double k2 = kx * kx + qy + qz;
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
            pi.scatter(b, put);
        }
        __syncthreads();
        ct_fft_range<N, true, true, NBF, SyncCta, PosTile, 1, L, false>(col, b, on, tw, none, put);

        fence_proxy_async();                             // my tile writes -> visible to the TMA store
        __syncthreads();
        if (tid == 0) {
            const int c0 = (first + it * stride) * (2 * TILE_COLS);
            for (int r0 = 0; r0 < N; r0 += W.box_rows) tma_store_3d(&tmap, c0, r0, 0, tile + (size_t)r0 * TILE_COLS);
            tma_store_commit();
        }
    }
    if (tid == 0) tma_store_wait<0>();
}

}  // namespace dgpe
