// xyfft_pair.cuh -- K2 / K4 / K3 on the TMA pipeline with TWO tiles in different phases per SM.
//
// k_fft_tma (xyfft_tma.cuh) keeps one CTA of N/8*8 threads per SM: its 16 warps all stop at every barrier between the
// passes of a tile (ncu: 7.5 warps stalled on `barrier` per issue, fp64 pipe 27 %), and a second CTA does not fit beside
// three 64 KB stages.  Here ONE CTA holds two independent teams ("halves") of xy_threads<N>() threads; each half walks
// every second tile of the CTA's sequence, synchronises on its own named barrier (bar.sync id, count), and the three
// shared-memory stages are shared: tile t lives in stage t % 3, so at any time two stages are being transformed -- by
// halves that drift into different phases, one computing while the other waits at a barrier or on shared memory -- and
// the third is in flight (the TMA store of a finished tile, then the TMA load of the tile three further on).
// The leader of the half that finished tile t-2 refills that stage with tile t+1 (which the OTHER half will consume)
// once its store has been read; arrival is signalled on the stage's mbarrier as in k_fft_tma.
//
// COLS = lines per tile (8: 128-byte rows).  Used at N = 512.  At N = 768 two teams of 8-line tiles would need 1536
// threads; with COLS = 4 (64-byte rows) the TMA moves the tiles five times slower (measured), and
// N = 384, 480 (radix-3/5 passes) spill 1-2 KB per thread inside the 64-register budget of a 1024-thread CTA.
// Constraints: 2 COLS N / rmax(N) <= 1024 threads, NSTAGE N COLS 16 bytes <= 227 KB, <= 64 registers per butterfly.
#pragma once
#include "xyfft_tma.cuh"

namespace dgpe {

template <int THREADS>
struct SyncHalf {
    static __device__ __forceinline__ void sync()
    {
        asm volatile("bar.sync %0, %1;\n" ::"r"(1 + (int)(threadIdx.x / THREADS)), "n"(THREADS) : "memory");
    }
};

// KIND = FFT_FWD / FFT_INV: transform along y, tensor map {2 (nz/2+1), ny, nx}; KIND = FFT_X_UDD: FFT along x, Udd~(k)/N,
// inverse FFT along x, tensor map {2 ny (nz/2+1), nx, 1} (as k_fft_tma / k_fft_tma_xudd).
template <int COLS>
struct PosCols {
    static __device__ __forceinline__ int at(int idx) { return idx * COLS; }
};
template <int N, int COLS>
__host__ __device__ constexpr int pair_team_threads() { return (COLS * xy_nbf<N>() + 31) / 32 * 32; }

// grid = min(ntiles, #SMs); block = 2 pair_team_threads<N, COLS>(); dynamic smem = NSTAGE N COLS 16 bytes (+128)
// W.tiles_per_batch / W.ntiles count tiles of COLS lines.
template <int N, int KIND, int COLS, int NSTAGE>
__global__ void __launch_bounds__(2 * pair_team_threads<N, COLS>(), 1)
k_fft_pair(const __grid_constant__ CUtensorMap tmap, TmaWalk W, const cplx* __restrict__ tw, UddArgs U, int ncols)
{
    constexpr int HT = pair_team_threads<N, COLS>();
    constexpr int NBF = xy_nbf<N>();
    constexpr int L = ct::npass(N);
    constexpr bool INV = KIND == FFT_INV;
    using PosTile = PosCols<COLS>;
    using Sync = SyncHalf<HT>;
    static_assert(L >= 2 && 2 * HT <= 1024, "two halves of a CTA");
    extern __shared__ unsigned char smem_dyn[];
    __shared__ __align__(8) unsigned long long full[NSTAGE];
    cplx* stages = reinterpret_cast<cplx*>(smem_dyn + ((128u - (smem_addr(smem_dyn) & 127u)) & 127u));
    constexpr int tile_elems = N * COLS;
    constexpr unsigned tile_bytes = (unsigned)tile_elems * 16u;
    const int half = threadIdx.x / HT, tid = threadIdx.x - half * HT, c = tid % COLS, b = tid / COLS;
    const bool on = b < NBF;
    const int first = blockIdx.x, stride = gridDim.x;
    const int nmine = (first < W.ntiles) ? (W.ntiles - first + stride - 1) / stride : 0;

    auto coords = [&](int it, int& c0, int& c2) {
        const int t = first + it * stride;
        if constexpr (KIND == FFT_X_UDD) {
            c0 = t * (2 * COLS);
            c2 = 0;
        } else {
            const int bat = t / W.tiles_per_batch;
            c0 = (t - bat * W.tiles_per_batch) * (2 * COLS);
            c2 = bat;
        }
    };
    auto issue_load = [&](int it) {                     // one thread
        int c0, c2;
        coords(it, c0, c2);
        const int st = it % NSTAGE;
        mbar_expect_tx(&full[st], tile_bytes);
        for (int r0 = 0; r0 < N; r0 += W.box_rows)
            tma_load_3d(stages + (size_t)st * tile_elems + (size_t)r0 * COLS, &tmap, c0, r0, c2, &full[st]);
    };

    if (threadIdx.x == 0) {
        for (int st = 0; st < NSTAGE; ++st) mbar_init(&full[st], 1);
        mbar_fence_init();
    }
    __syncthreads();
    if (threadIdx.x == 0)
        for (int it = 0; it < NSTAGE && it < nmine; ++it) issue_load(it);

    auto none = [](int) { return mk(0.0, 0.0); };
    for (int it = half; it < nmine; it += 2) {
        const int st = it % NSTAGE;
        cplx* tile = stages + (size_t)st * tile_elems;
        cplx* col = tile + c;
        auto put = [&](int idx, cplx val) { col[PosTile::at(idx)] = val; };
        double qy = 0.0, qz = 0.0;
        if constexpr (KIND == FFT_X_UDD) {
            // ky^2, kz^2 of this thread's column (columns past the end of a ragged last tile take the last column's)
            const int cidx = min((first + it * stride) * COLS + c, ncols - 1);
            const int ky = cidx / U.nzh, kz = cidx - ky * U.nzh;
            qy = __ldg(&U.ky2[ky]);
            qz = __ldg(&U.kz2[kz]);
        }
        mbar_wait(&full[st], (unsigned)((it / NSTAGE) & 1));

        // pass 0 by hand: after its barrier this half's leader refills the stage of the half's previous tile (it - 2),
        // which is the stage of tile it - 2 + NSTAGE (with three stages: the other half's next tile)
        CtPass<N, 0, INV, false, NBF> p0;
        if (on) {
            if constexpr (KIND == FFT_X_UDD) p0.load_tw(b, tw);
            p0.load(b, [&](int idx) { return col[PosTile::at(idx)]; });
        }
        Sync::sync();                                    // every read of pass 0 precedes its writes
        if (tid == 0 && it >= 2 && it - 2 + NSTAGE < nmine) {
            tma_store_wait_read<0>();                    // my store of tile it - 2 has read its stage
            issue_load(it - 2 + NSTAGE);
        }
        if (on) {
            p0.bfly(b);
            p0.scatter(b, put);
        }
        if constexpr (KIND != FFT_X_UDD) {
            CtPass<N, 1, INV, false, NBF> p1;
            if (on) p1.load_tw(b, tw);                   // overlaps the barrier wait
            Sync::sync();
            ct_fft_range_tw<N, INV, false, NBF, Sync, PosTile, 1, L, false>(p1, col, b, on, tw, none, put);
        } else {
            if constexpr (L > 2) {
                CtPass<N, 1, false, false, NBF> p1;
                if (on) p1.load_tw(b, tw);
                Sync::sync();
                ct_fft_range_tw<N, false, false, NBF, Sync, PosTile, 1, L - 1, false>(p1, col, b, on, tw, none, put);
            } else {
                Sync::sync();
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
            Sync::sync();
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
                    if (k2 == 0.0) u = 0.0;              // Udd~(0) = 0 (R#11)
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
            Sync::sync();
            ct_fft_range<N, true, true, NBF, Sync, PosTile, 1, L, false>(col, b, on, tw, none, put);
        }

        fence_proxy_async();                             // my tile writes -> visible to the TMA store
        Sync::sync();
        if (tid == 0) {
            int c0, c2;
            coords(it, c0, c2);
            for (int r0 = 0; r0 < N; r0 += W.box_rows) tma_store_3d(&tmap, c0, r0, c2, tile + (size_t)r0 * COLS);
            tma_store_commit();
        }
    }
    if (tid == 0) tma_store_wait<0>();
}

}  // namespace dgpe
