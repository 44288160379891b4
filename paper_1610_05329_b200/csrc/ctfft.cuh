// ctfft.cuh -- compile-time-planned Stockham passes whose butterflies live in registers, used by the
// specialised kernels in xyfft.cuh (strided axes x, y) and zline.cuh (contiguous axis z).
//
// Same mathematics as fft.cuh (P:L130 FFT-friendly sizes 2^a 3^b; BJ:north_star "mixed-radix
// (2^a 3^b) shared-memory Stockham FFT passes per axis"): pass p with radix R and Ns = product of the
// radices before it computes, for every butterfly j in [0, N/R), k = j mod Ns,
//     v_q = in[j + q N/R] w_N^{q k N/(Ns R)},    out[(j div Ns) Ns R + k + s Ns] = sum_q v_q w_R^{q s}.
// Here N and the radix sequence are template constants, so every index folds at compile time and a
// thread keeps its butterflies in registers between the read side and the write side of a pass.
// The radix sequence is 8.., 4, 2, 3.., 5.., 7.. (REV = false) or its reverse (REV = true).  With the reversed
// sequence the first pass of a transform reads exactly the elements the last pass of a forward-order
// transform produced in the same thread, so a forward and an inverse transform chain in registers
// (K3: FFT_x, multiply by Udd~(k), IFFT_x -- BJ:north_star).
#pragma once
#include "fft.cuh"

namespace dgpe {
namespace ct {

__host__ __device__ constexpr int pick(int m)
{
    return (m % 8 == 0) ? 8 : (m % 4 == 0) ? 4 : (m % 2 == 0) ? 2 : (m % 3 == 0) ? 3 : (m % 5 == 0) ? 5 : 7;
}
// Lengths whose plan starts with a radix other than pick()'s: n/32 for the z-line transforms of nz = 192,
// 320, 384 (M = 96, 160, 192), so that their first pass is one butterfly per lane, fed from registers
// with every lane busy (zline.cuh).  Any radix order is a valid transform; the x/y kernels of the same
// lengths simply use the same plan.
// (250 = nz/2 at nz = 500: radix 5 first gives 50 butterflies, two per lane, instead of 125 of radix 2)
__host__ __device__ constexpr int first_of(int n) { return n == 192 ? 6 : n == 160 ? 5 : n == 96 ? 3 : n == 250 ? 5 : 0; }
__host__ __device__ constexpr int npass(int n)
{
    int c = 0;
    if (first_of(n)) { n /= first_of(n); ++c; }
    while (n > 1) { n /= pick(n); ++c; }
    return c;
}
__host__ __device__ constexpr int radix_fwd(int n, int p)
{
    if (first_of(n)) {
        if (p == 0) return first_of(n);
        n /= first_of(n);
        --p;
    }
    for (int i = 0; i < p; ++i) n /= pick(n);
    return pick(n);
}
__host__ __device__ constexpr int radix_at(int n, int p, bool rev) { return radix_fwd(n, rev ? npass(n) - 1 - p : p); }
__host__ __device__ constexpr int ns_at(int n, int p, bool rev)
{
    int ns = 1;
    for (int i = 0; i < p; ++i) ns *= radix_at(n, i, rev);
    return ns;
}
__host__ __device__ constexpr int rmax(int n)
{
    int r = 1;
    if (first_of(n)) { r = first_of(n); n /= r; }
    while (n > 1) { int q = pick(n); if (q > r) r = q; n /= q; }
    return r;
}
}  // namespace ct

// Pass P of an N-point transform for a team of NBF butterfly slots (slot b handles butterflies
// b, b + NBF, ...).  load -> (barrier, if the passes run in place) -> bfly -> scatter.
template <int N, int P, bool INV, bool REV, int NBF>
struct CtPass {
    static constexpr int R = ct::radix_at(N, P, REV);
    static constexpr int Ns = ct::ns_at(N, P, REV);
    static constexpr int NBUT = N / R;
    static constexpr int NB = (NBUT + NBF - 1) / NBF;
    static constexpr bool EXACT = (NBUT % NBF) == 0;
    static constexpr int TWSTEP = N / (Ns * R);
    static constexpr int NPASS = ct::npass(N);
    static constexpr bool LAST = (P == NPASS - 1);

    cplx v[NB][R];
    cplx w[Ns > 1 ? NB : 1][R];      // twiddles w^q of this slot's butterflies (unused when Ns == 1)

    // Twiddles w^q, w = tw[k TWSTEP] (tw[m] = exp(-2 pi i m/N)): the powers 1, 2, 4 come from the fp64
    // table, the others are one product of two table entries (<= 3 ulp), which trades 4 of the 7 table
    // loads of a radix-8 butterfly for 4 complex multiplications.  Independent of the data, so callers
    // issue it BEFORE the barrier that guards the data: the table loads overlap the barrier wait.
    __device__ __forceinline__ void load_tw(int b, const cplx* __restrict__ tw)
    {
        if constexpr (Ns > 1) {
#pragma unroll
            for (int u = 0; u < NB; ++u) {
                const int j = b + u * NBF;
                if (EXACT || j < NBUT) {
                    const int k = j % Ns;
#pragma unroll
                    for (int q = 1; q < R; q <<= 1) {
                        w[u][q] = __ldg(&tw[q * k * TWSTEP]);
                        if (INV) w[u][q].y = -w[u][q].y;
                    }
                }
            }
        }
    }

    // v_q = f(j + q N/R) w^q for this slot's butterflies (load_tw first)
    template <class F>
    __device__ __forceinline__ void load(int b, F&& f)
    {
#pragma unroll
        for (int u = 0; u < NB; ++u) {
            const int j = b + u * NBF;
            if (EXACT || j < NBUT) {
#pragma unroll
                for (int q = 0; q < R; ++q) v[u][q] = f(j + q * NBUT);
                if constexpr (Ns > 1) {
                    if constexpr (R >= 4) w[u][3] = cmul(w[u][1], w[u][2]);
                    if constexpr (R >= 6) w[u][5] = cmul(w[u][1], w[u][4]);
                    if constexpr (R >= 7) w[u][6] = cmul(w[u][2], w[u][4]);
                    if constexpr (R >= 8) w[u][7] = cmul(w[u][3], w[u][4]);
#pragma unroll
                    for (int q = 1; q < R; ++q) v[u][q] = cmul(v[u][q], w[u][q]);
                }
            }
        }
    }

    __device__ __forceinline__ void bfly(int b)
    {
#pragma unroll
        for (int u = 0; u < NB; ++u) {
            const int j = b + u * NBF;
            if (EXACT || j < NBUT) Butterfly<R, INV>::run(v[u]);
        }
    }

    // f(output index, value) for every output of this slot; for_each may also rewrite v in place
    template <class F>
    __device__ __forceinline__ void scatter(int b, F&& f)
    {
#pragma unroll
        for (int u = 0; u < NB; ++u) {
            const int j = b + u * NBF;
            if (EXACT || j < NBUT) {
                const int k = j % Ns;
                const int base = (j / Ns) * Ns * R + k;
#pragma unroll
                for (int s = 0; s < R; ++s) f(base + s * Ns, v[u][s]);
            }
        }
    }
    template <class F>
    __device__ __forceinline__ void modify(int b, F&& f)     // v <- f(output index, v)
    {
#pragma unroll
        for (int u = 0; u < NB; ++u) {
            const int j = b + u * NBF;
            if (EXACT || j < NBUT) {
                const int k = j % Ns;
                const int base = (j / Ns) * Ns * R + k;
#pragma unroll
                for (int s = 0; s < R; ++s) v[u][s] = f(base + s * Ns, v[u][s]);
            }
        }
    }
};

// Barrier between the passes of one team: the whole CTA (strided-axis tiles) or one warp (z lines).
struct SyncCta { static __device__ __forceinline__ void sync() { __syncthreads(); } };
struct SyncWarp { static __device__ __forceinline__ void sync() { __syncwarp(); } };

// Passes P .. PEND-1 of an N-point transform, in place in a shared-memory column: element idx of the
// column lives at col[Pos::at(idx)].  Pass P takes its inputs from `first(idx)` if FROM_F (else from
// the column).  The final pass of the transform (P = NPASS-1) hands its outputs to `last(idx, value)`;
// every other pass writes the column and ends with a team barrier.
// `on` = this thread owns butterfly slot b (threads that do not still take part in the barriers).
// When FROM_F is false the caller must have synchronised the team after the column was written; when
// it is true the column must be free to overwrite.
// worker: the twiddles of pass P are already in `pass` (loaded before the preceding barrier)
template <int N, bool INV, bool REV, int NBF, class Sync, class Pos, int P, int PEND, bool FROM_F, class FFirst,
          class FLast>
__device__ __forceinline__ void ct_fft_range_tw(CtPass<N, P, INV, REV, NBF>& pass, cplx* col, int b, bool on,
                                                const cplx* __restrict__ tw, FFirst&& first, FLast&& last)
{
    using Pass = CtPass<N, P, INV, REV, NBF>;
    if (on) {
        if constexpr (FROM_F) pass.load(b, first);
        else pass.load(b, [&](int idx) { return col[Pos::at(idx)]; });
    }
    if constexpr (!FROM_F) Sync::sync();          // every read of this pass precedes its writes
    if (on) pass.bfly(b);
    if constexpr (Pass::LAST) {
        if (on) pass.scatter(b, last);
    } else {
        if (on) pass.scatter(b, [&](int idx, cplx val) { col[Pos::at(idx)] = val; });
        if constexpr (P + 1 < PEND) {
            CtPass<N, P + 1, INV, REV, NBF> next;
            if (on) next.load_tw(b, tw);          // overlaps the barrier wait
            Sync::sync();
            ct_fft_range_tw<N, INV, REV, NBF, Sync, Pos, P + 1, PEND, false>(next, col, b, on, tw, first, last);
        } else {
            Sync::sync();
        }
    }
}

template <int N, bool INV, bool REV, int NBF, class Sync, class Pos, int P, int PEND, bool FROM_F, class FFirst,
          class FLast>
__device__ __forceinline__ void ct_fft_range(cplx* col, int b, bool on, const cplx* __restrict__ tw, FFirst&& first,
                                             FLast&& last)
{
    if constexpr (P < PEND) {
        CtPass<N, P, INV, REV, NBF> pass;
        if (on) pass.load_tw(b, tw);
        ct_fft_range_tw<N, INV, REV, NBF, Sync, Pos, P, PEND, FROM_F>(pass, col, b, on, tw, first, last);
    }
}

// ---- streaming global accesses (every array of the step is far larger than L2) ----
__device__ __forceinline__ cplx ld_stream(const cplx* p)
{
    cplx v;
    asm volatile("ld.global.cs.v2.f64 {%0, %1}, [%2];\n" : "=d"(v.x), "=d"(v.y) : "l"(p));
    return v;
}
__device__ __forceinline__ double ld_stream(const double* p)
{
    double v;
    asm volatile("ld.global.cs.f64 %0, [%1];\n" : "=d"(v) : "l"(p));
    return v;
}
__device__ __forceinline__ void st_stream(cplx* p, cplx v)
{
    asm volatile("st.global.cs.v2.f64 [%0], {%1, %2};\n" ::"l"(p), "d"(v.x), "d"(v.y) : "memory");
}

// L2 prefetch of the 128-byte line holding p: kernels ask for the data of the tile / line that will be
// processed one "residency" later, so that the demand loads of that later CTA hit L2 instead of HBM
__device__ __forceinline__ void prefetch_l2(const void* p) { asm volatile("prefetch.global.L2 [%0];\n" ::"l"(p)); }

}  // namespace dgpe
