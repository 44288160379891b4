// xyfft_fused.cuh -- K2, K3 and K4 as ONE launch whose intermediate results never leave L2
// (SV section 8a rows a2-a4; BJ:north_star "mixed-radix shared-memory Stockham FFT passes per axis", "Udd(k)
// multiply fused into the forward-last and inverse-first passes").
//
// The three middle passes of the dipolar convolution -- FFT along y, FFT along x . Udd~(k)/N . inverse FFT along
// x, inverse FFT along y -- touch one kz-SLAB of the half-spectrum (8 neighbouring kz bins x all ky x all kx:
// nx ny 128 bytes, 33.5 MB at 512^2) independently of every other slab.  As three launches each of them streams
// the whole half-spectrum S through HBM (6 S bytes); here one launch walks the slabs, so a slab is read from HBM
// once by the y pass (phase A), stays in the 126 MB L2 while the x pass (phase B) and the inverse y pass (phase C)
// work on it in place, and goes back to HBM once: 2 S bytes.
//
// Work items = tiles (8 lines x the whole line, exactly the tiles and the register/shared-memory passes of
// k_fft_xy in xyfft.cuh), one CTA per tile.  A CTA takes the next tile of a queue (an atomic counter) when it
// starts, so tiles begin in queue order.  The queue interleaves the phases of neighbouring slab groups,
//        A(g), C(g-1), B(g), A(g+1), C(g), B(g+1), ...
// so that the phase a tile depends on was handed out a whole phase earlier: B(g) tiles need every A tile of their
// slab finished, C(g) tiles every B tile; a tile waits on its slab's counter (acquire), and announces itself on
// it (release) when its stores are done.  Two groups are alive in L2 at a time.  A CTA only ever waits for
// tiles that were claimed before its own, and a claimed tile is held by a running CTA, so the queue cannot
// deadlock whatever the number of resident CTAs or the order in which the hardware dispatches them.
// (A persistent loop over the tiles in one CTA costs the 64-register budget of two resident 512-thread CTAs
// ~2.5 KB of spills per thread; one CTA per tile compiles without any.)
//
// nx == ny == N (every BASELINE config and every grid of the paper's tables); other shapes use the three
// separate kernels.
#pragma once
#include "xyfft.cuh"

namespace dgpe {

struct FusedWalk {
    int ny, nzh;                // lines along y per x plane, kz bins per row
    int nslab;                  // kz slabs = ceil(nzh / 8)
    int nunits;                 // (phase, slab) units in queue order = 3 nslab
    const int* units;           // unit -> phase (bits 0-1: 0 = A, 1 = B, 2 = C) | slab << 2
    unsigned int* head;         // queue head
    unsigned int* done;         // [2][nslab]: finished tiles of phase A, of phase B
    int pf_items;               // L2 prefetch of the phase-A tile this many queue items ahead; 0 = off
};

__device__ __forceinline__ unsigned int ld_acquire_gpu(const unsigned int* p)
{
    unsigned int v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];\n" : "=r"(v) : "l"(p) : "memory");
    return v;
}
// L2-only accesses with the default replacement policy: the slab is to stay in L2 between the phases
__device__ __forceinline__ cplx ld_l2(const cplx* p)
{
    cplx v;
    asm volatile("ld.global.cg.v2.f64 {%0, %1}, [%2];\n" : "=d"(v.x), "=d"(v.y) : "l"(p));
    return v;
}
__device__ __forceinline__ void st_l2(cplx* p, cplx v)
{
    asm volatile("st.global.cg.v2.f64 [%0], {%1, %2};\n" ::"l"(p), "d"(v.x), "d"(v.y) : "memory");
}

// One tile of phase A (INV = false: forward FFT along y, results stay in L2) or phase C (INV = true: inverse FFT
// along y, results stream out to HBM).  Separate functions (not inlined) so that each phase gets the register
// allocation of the stand-alone kernel it came from; the persistent loop around them holds almost no state.
template <int N, bool INV>
__device__ __forceinline__ void fused_tile_y(cplx* g, long long es, cplx* colsm, int b, bool on, const cplx* __restrict__ tw)
{
    constexpr int NBF = xy_nbf<N>();
    constexpr int L = ct::npass(N);
    auto from_g = [&](int idx) { return ld_l2(g + (long long)idx * es); };
    if constexpr (!INV) {
        auto to_g = [&](int idx, cplx v) { st_l2(g + (long long)idx * es, v); };
        ct_fft_range<N, false, false, NBF, SyncCta, PosTile, 0, L, true>(colsm, b, on, tw, from_g, to_g);
    } else {
        auto to_g = [&](int idx, cplx v) { st_stream(g + (long long)idx * es, v); };
        ct_fft_range<N, true, false, NBF, SyncCta, PosTile, 0, L, true>(colsm, b, on, tw, from_g, to_g);
    }
}

// One tile of phase B: FFT along x, Udd~(k)/N, inverse FFT along x (as k_fft_xy<N, FFT_X_UDD>), in L2.
template <int N>
__device__ __forceinline__ void fused_tile_x(cplx* g, long long es, cplx* colsm, int b, bool on, const cplx* __restrict__ tw,
                                          double qy, double qz, bool origin_col, double dkx, double invN)
{
    constexpr int NBF = xy_nbf<N>();
    constexpr int L = ct::npass(N);
    auto from_g = [&](int idx) { return ld_l2(g + (long long)idx * es); };
    auto to_g = [&](int idx, cplx v) { st_l2(g + (long long)idx * es, v); };
    ct_fft_range<N, false, false, NBF, SyncCta, PosTile, 0, L - 1, true>(colsm, b, on, tw, from_g, to_g);
    // last forward pass, Udd~(k)/N, first inverse pass: one set of registers
    using PF = CtPass<N, L - 1, false, false, NBF>;
    using PI = CtPass<N, 0, true, true, NBF>;
    static_assert(PF::R == PI::R && PF::NB == PI::NB && PI::Ns == 1, "forward-last and inverse-first passes must match");
    PF pf;
    if (on) {
        pf.load_tw(b, tw);
        pf.load(b, [&](int idx) { return colsm[PosTile::at(idx)]; });
    }
    __syncthreads();
    PI pi;
    if (on) {
        pf.bfly(b);
        // Udd~(k) = (4 pi/3)(3 kz^2/|k|^2 - 1), Udd~(0) = 0 (BJ:configs[0]; R#11)
        const double FOUR_PI_3 = 4.1887902047863909846168578443727;
        pf.modify(b, [&](int idx, cplx v) {
            const double kx = (double)(idx <= N / 2 ? idx : idx - N) * dkx;
            const double k2 = kx * kx + qy + qz;
            double rk = (double)__frcp_rn((float)k2);
            rk = rk * (2.0 - k2 * rk);
            rk = rk * (2.0 - k2 * rk);
            double u = FOUR_PI_3 * (3.0 * qz * rk - 1.0);
            if (origin_col && idx == 0) u = 0.0;
            u *= invN;
            return mk(v.x * u, v.y * u);
        });
#pragma unroll
        for (int u = 0; u < PF::NB; ++u)
#pragma unroll
            for (int q = 0; q < PF::R; ++q) pi.v[u][q] = pf.v[u][q];
        pi.bfly(b);
        pi.scatter(b, [&](int idx, cplx val) { colsm[PosTile::at(idx)] = val; });
    }
    __syncthreads();
    ct_fft_range<N, true, true, NBF, SyncCta, PosTile, 1, L, false>(colsm, b, on, tw, from_g, to_g);
}

// grid = number of tiles (3 nslab N); block = xy_threads<N>(); dynamic shared memory = N*128 bytes.
// A CTA takes the next tile of the queue (not blockIdx: the order of the claims is then the order in which CTAs
// start, whatever order the hardware dispatches them in).
template <int N>
__global__ void __launch_bounds__(xy_threads<N>(), xy_min_ctas<N>())
k_fft_yxy(cplx* __restrict__ spec, FusedWalk W, const cplx* __restrict__ tw, UddArgs U)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ unsigned int s_item;
    constexpr int NBF = xy_nbf<N>();
    static_assert(ct::npass(N) >= 2, "the fused kernel is for lines of at least two passes");
    const int tid = threadIdx.x, c = tid & 7, b = tid >> 3;
    if (tid == 0) s_item = atomicAdd(W.head, 1u);
    __syncthreads();
    const unsigned int item = s_item;
    const int unit = (int)(item / N), t = (int)(item - (unsigned int)unit * N);
    const int code = __ldg(&W.units[unit]);
    const int phase = code & 3, slab = code >> 2;
    const int kz = slab * TILE_COLS + c;
    const bool colok = kz < W.nzh;
    const bool on = colok && b < NBF;
    const long long row = W.nzh, plane = (long long)W.ny * W.nzh;
    cplx* colsm = reinterpret_cast<cplx*>(smem_raw) + c;

    if (phase != 0) {
        if (tid == 0) {
            const unsigned int* d = W.done + (phase == 1 ? 0 : W.nslab) + slab;
            while (ld_acquire_gpu(d) < (unsigned int)N) __nanosleep(40);
        }
        __syncthreads();
    } else if (W.pf_items > 0) {
        // ask L2 for the phase-A tile (HBM) that is W.pf_items further down the queue
        const unsigned int it2 = item + (unsigned int)W.pf_items;
        if (it2 < (unsigned int)W.nunits * N) {
            const int u2 = (int)(it2 / N), t2 = (int)(it2 - (unsigned int)u2 * N);
            const int code2 = __ldg(&W.units[u2]);
            if ((code2 & 3) == 0) {
                const char* t0 = reinterpret_cast<const char*>(spec + (long long)t2 * plane + (code2 >> 2) * TILE_COLS);
                for (int j = tid; j < 2 * N; j += xy_threads<N>())
                    prefetch_l2(t0 + (long long)(j >> 1) * row * 16 + (j & 1) * 112);
            }
        }
    }

    if (phase == 0) {
        // A / C: lines along y of x plane t; element j of column kz at spec[(t ny + j) nzh + kz]
        fused_tile_y<N, false>(spec + (long long)t * plane + (colok ? kz : 0), row, colsm, b, on, tw);
    } else if (phase == 2) {
        fused_tile_y<N, true>(spec + (long long)t * plane + (colok ? kz : 0), row, colsm, b, on, tw);
        return;
    } else {
        // B: lines along x at ky = t; element i of column kz at spec[(i ny + t) nzh + kz]
        fused_tile_x<N>(spec + (long long)t * row + (colok ? kz : 0), plane, colsm, b, on, tw, __ldg(&U.ky2[t]),
                        __ldg(&U.kz2[colok ? kz : 0]), t == 0 && kz == 0, U.dkx, U.invN);
    }
    __syncthreads();            // every store of this tile is issued
    if (threadIdx.x == 0) {
        __threadfence();        // release: the CTA's stores (ordered before by the barrier) are visible gpu-wide
        atomicAdd(W.done + (phase == 0 ? 0 : W.nslab) + slab, 1u);
    }
}

}  // namespace dgpe
