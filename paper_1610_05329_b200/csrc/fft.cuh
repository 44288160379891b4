// fft.cuh -- mixed-radix (2, 3, 4, 5, 7, 8, 11, 13) Stockham autosort FFT passes over a shared-memory tile of
// TILE_COLS lines (FFT-friendly sizes 2^a 3^b 5^c 7^d ...; BJ:north_star "mixed-radix (2^a 3^b)
// shared-memory Stockham FFT passes per axis").
//
// Pass p of an n-point transform with radix R and Ns = product of the radices of the passes before it:
//   for every butterfly j in [0, n/R):   k = j mod Ns
//     v_q  = in[j + q n/R] * w_n^{q k n/(Ns R)}                 q = 0..R-1
//     out[(j div Ns) Ns R + k + s Ns] = sum_q v_q w_R^{q s}     s = 0..R-1
// w_n = exp(-2 pi i/n) forward, exp(+2 pi i/n) inverse; no normalisation.
//
// Thread layout: thread = (c, b), c = tid & 7 the tile column (line), b = tid >> 3 the butterfly slot.
// A quarter-warp (8 lanes, one 128-byte shared-memory wavefront of a 16-byte access) is the 8 columns
// of ONE tile row, so every access pattern along the transform index is bank-conflict free.
// Passes run in place: each thread holds its NB butterflies (NB*R values) in registers across the
// barrier that separates the reads of a pass from its writes.
#pragma once
#include "common.cuh"

namespace dgpe {

template <bool INV>
__device__ __forceinline__ cplx mul_w4(cplx a)   // * w_4 = -i (forward) or +i (inverse)
{
    return INV ? mul_pi(a) : mul_mi(a);
}

template <int R, bool INV>
struct Butterfly;

template <bool INV>
struct Butterfly<2, INV> {
    static __device__ __forceinline__ void run(cplx (&v)[2])
    {
        cplx a = v[0], b = v[1];
        v[0] = cadd(a, b);
        v[1] = csub(a, b);
    }
};

template <bool INV>
struct Butterfly<3, INV> {
    static __device__ __forceinline__ void run(cplx (&v)[3])
    {
        const double S = 0.86602540378443864676372317075294;   // sin(pi/3)
        cplx t1 = cadd(v[1], v[2]);
        cplx m1 = mk(v[0].x - 0.5 * t1.x, v[0].y - 0.5 * t1.y);
        cplx df = cscale(csub(v[1], v[2]), S);
        cplx m2 = mul_w4<INV>(df);                              // -i S (v1 - v2) forward
        v[0] = cadd(v[0], t1);
        v[1] = cadd(m1, m2);
        v[2] = csub(m1, m2);
    }
};

// Odd prime radix R = 2h+1 (5, 7, 11, 13: P:L130 lists 2^a 3^b 5^c 7^d 11^e 13^f as the FFT-friendly sizes): with
// a_k = v_k + v_{R-k}, b_k = v_k - v_{R-k}  (k = 1..h)
//   out_s, out_{R-s} = (v_0 + sum_k cos(2 pi s k/R) a_k)  -/+  i sum_k sin(2 pi s k/R) b_k   (forward; signs swap for the inverse)
template <int R, bool INV>
struct OddPrimeButterfly {
    static __device__ __forceinline__ void run(cplx (&v)[R], const double (&C)[R], const double (&S)[R])
    {
        constexpr int H = (R - 1) / 2;
        cplx a[H], b[H];
#pragma unroll
        for (int k = 1; k <= H; ++k) {
            a[k - 1] = cadd(v[k], v[R - k]);
            b[k - 1] = csub(v[k], v[R - k]);
        }
        cplx sum = v[0];
#pragma unroll
        for (int k = 0; k < H; ++k) sum = cadd(sum, a[k]);
        cplx out[R];
        out[0] = sum;
#pragma unroll
        for (int s = 1; s <= H; ++s) {
            cplx re = v[0], im = mk(0.0, 0.0);
#pragma unroll
            for (int k = 1; k <= H; ++k) {
                const int m = (s * k) % R;
                re = mk(fma(C[m], a[k - 1].x, re.x), fma(C[m], a[k - 1].y, re.y));
                im = mk(fma(S[m], b[k - 1].x, im.x), fma(S[m], b[k - 1].y, im.y));
            }
            const cplx t = mul_w4<INV>(im);              // -i im (forward), +i im (inverse)
            out[s] = cadd(re, t);
            out[R - s] = csub(re, t);
        }
#pragma unroll
        for (int s = 0; s < R; ++s) v[s] = out[s];
    }
};

template <bool INV>
struct Butterfly<5, INV> {
    static __device__ __forceinline__ void run(cplx (&v)[5])
    {
        // cos, sin of 2 pi m/5
        const double C[5] = {1.0, 0.30901699437494742410229341718282, -0.80901699437494742410229341718282,
                             -0.80901699437494742410229341718282, 0.30901699437494742410229341718282};
        const double S[5] = {0.0, 0.95105651629515357211643933337938, 0.58778525229247312916870595463907,
                             -0.58778525229247312916870595463907, -0.95105651629515357211643933337938};
        OddPrimeButterfly<5, INV>::run(v, C, S);
    }
};

template <bool INV>
struct Butterfly<7, INV> {
    static __device__ __forceinline__ void run(cplx (&v)[7])
    {
        // cos, sin of 2 pi m/7
        const double C[7] = {1.0, 0.62348980185873353052500488400424, -0.22252093395631440428890256449679,
                             -0.90096886790241912623610231950745, -0.90096886790241912623610231950745,
                             -0.22252093395631440428890256449679, 0.62348980185873353052500488400424};
        const double S[7] = {0.0, 0.78183148246802980870844452667406, 0.97492791218182360701813168299393,
                             0.43388373911755812047576833284836, -0.43388373911755812047576833284836,
                             -0.97492791218182360701813168299393, -0.78183148246802980870844452667406};
        OddPrimeButterfly<7, INV>::run(v, C, S);
    }
};

template <bool INV>
struct Butterfly<11, INV> {
    static __device__ __forceinline__ void run(cplx (&v)[11])
    {
        // cos, sin of 2 pi m/11
        const double C[11] = {1.0, 0.8412535328311812, 0.41541501300188644, -0.142314838273285, -0.654860733945285, -0.9594929736144974, -0.9594929736144975, -0.6548607339452852, -0.14231483827328523, 0.41541501300188605, 0.8412535328311812};
        const double S[11] = {0.0, 0.5406408174555976, 0.9096319953545183, 0.9898214418809328, 0.7557495743542583, 0.28173255684142967, -0.2817325568414294, -0.7557495743542582, -0.9898214418809327, -0.9096319953545186, -0.5406408174555974};
        OddPrimeButterfly<11, INV>::run(v, C, S);
    }
};

template <bool INV>
struct Butterfly<13, INV> {
    static __device__ __forceinline__ void run(cplx (&v)[13])
    {
        // cos, sin of 2 pi m/13
        const double C[13] = {1.0, 0.8854560256532099, 0.5680647467311559, 0.120536680255323, -0.35460488704253545, -0.7485107481711012, -0.970941817426052, -0.9709418174260521, -0.7485107481711013, -0.3546048870425359, 0.1205366802553232, 0.5680647467311548, 0.88545602565321};
        const double S[13] = {0.0, 0.4647231720437685, 0.8229838658936564, 0.992708874098054, 0.9350162426854148, 0.6631226582407952, 0.23931566428755768, -0.23931566428755743, -0.663122658240795, -0.9350162426854147, -0.992708874098054, -0.822983865893657, -0.4647231720437684};
        OddPrimeButterfly<13, INV>::run(v, C, S);
    }
};

template <bool INV>
struct Butterfly<4, INV> {
    static __device__ __forceinline__ void run(cplx (&v)[4])
    {
        cplx t0 = cadd(v[0], v[2]), t1 = csub(v[0], v[2]);
        cplx t2 = cadd(v[1], v[3]), t3 = mul_w4<INV>(csub(v[1], v[3]));
        v[0] = cadd(t0, t2);
        v[1] = cadd(t1, t3);
        v[2] = csub(t0, t2);
        v[3] = csub(t1, t3);
    }
};

// 6 = 2 x 3: two radix-3 butterflies on the even and the odd inputs, twiddles w_6^k, one radix-2 step
template <bool INV>
struct Butterfly<6, INV> {
    static __device__ __forceinline__ void run(cplx (&v)[6])
    {
        const double S = 0.86602540378443864676372317075294;   // sin(pi/3)
        cplx e[3] = {v[0], v[2], v[4]};
        cplx o[3] = {v[1], v[3], v[5]};
        Butterfly<3, INV>::run(e);
        Butterfly<3, INV>::run(o);
        // w_6 = 1/2 -/+ i S (forward / inverse), w_6^2 = -1/2 -/+ i S
        const cplx w1 = INV ? mk(0.5, S) : mk(0.5, -S), w2 = INV ? mk(-0.5, S) : mk(-0.5, -S);
        const cplx o1 = cmul(o[1], w1), o2 = cmul(o[2], w2);
        v[0] = cadd(e[0], o[0]);
        v[3] = csub(e[0], o[0]);
        v[1] = cadd(e[1], o1);
        v[4] = csub(e[1], o1);
        v[2] = cadd(e[2], o2);
        v[5] = csub(e[2], o2);
    }
};

template <bool INV>
struct Butterfly<8, INV> {
    static __device__ __forceinline__ void run(cplx (&v)[8])
    {
        const double H = 0.70710678118654752440084436210485;   // sqrt(1/2)
        cplx e[4] = {v[0], v[2], v[4], v[6]};
        cplx o[4] = {v[1], v[3], v[5], v[7]};
        Butterfly<4, INV>::run(e);
        Butterfly<4, INV>::run(o);
        // w_8^1 = (1 -/+ i)/sqrt2, w_8^2 = -/+ i, w_8^3 = (-1 -/+ i)/sqrt2   (forward / inverse)
        cplx o1 = INV ? mk((o[1].x - o[1].y) * H, (o[1].x + o[1].y) * H)
                      : mk((o[1].x + o[1].y) * H, (o[1].y - o[1].x) * H);
        cplx o2 = mul_w4<INV>(o[2]);
        cplx o3 = INV ? mk((-o[3].x - o[3].y) * H, (o[3].x - o[3].y) * H)
                      : mk((o[3].y - o[3].x) * H, (-o[3].x - o[3].y) * H);
        v[0] = cadd(e[0], o[0]);
        v[4] = csub(e[0], o[0]);
        v[1] = cadd(e[1], o1);
        v[5] = csub(e[1], o1);
        v[2] = cadd(e[2], o2);
        v[6] = csub(e[2], o2);
        v[3] = cadd(e[3], o3);
        v[7] = csub(e[3], o3);
    }
};

// One pass.  src/dst are generic pointers (shared or global) already offset to this thread's column;
// sstride/dstride = elements between consecutive transform indices.  `active` masks the columns of a
// ragged last tile; every thread of the block must call (two block barriers inside).
template <int R, int NB, bool INV>
__device__ __noinline__ void fft_pass(int n, int Ns, int b, int nbf, bool active,
                                         const cplx* src, long long sstride,
                                         cplx* dst, long long dstride,
                                         const cplx* __restrict__ tw)
{
    const int nbut = n / R;
    const int twstep = n / (Ns * R);
    cplx v[NB][R];
#pragma unroll
    for (int u = 0; u < NB; ++u) {
        const int j = b + u * nbf;
        if (active && j < nbut) {
            const int k = j % Ns;
#pragma unroll
            for (int q = 0; q < R; ++q) v[u][q] = src[(long long)(j + q * nbut) * sstride];
            if (Ns > 1) {
#pragma unroll
                for (int q = 1; q < R; ++q) {
                    cplx w = __ldg(&tw[q * k * twstep]);
                    if (INV) w.y = -w.y;
                    v[u][q] = cmul(v[u][q], w);
                }
            }
        }
    }
    __syncthreads();
#pragma unroll
    for (int u = 0; u < NB; ++u) {
        const int j = b + u * nbf;
        if (active && j < nbut) {
            Butterfly<R, INV>::run(v[u]);
            const int k = j % Ns;
            const int base = (j / Ns) * Ns * R + k;
#pragma unroll
            for (int s = 0; s < R; ++s) dst[(long long)(base + s * Ns) * dstride] = v[u][s];
        }
    }
    __syncthreads();
}

// All passes of one transform.  The first pass reads `src` (stride sstride), the last writes `dst`
// (stride dstride); everything in between goes through the shared-memory tile `sm` (stride smstride).
// src and/or dst may be the tile itself.
template <bool INV>
__device__ __forceinline__ void fft_run(const FftPlan& P, int b, bool active,
                                        const cplx* src, long long sstride,
                                        cplx* sm, long long smstride,
                                        cplx* dst, long long dstride)
{
    int Ns = 1;
    for (int p = 0; p < P.npass; ++p) {
        const cplx* s = (p == 0) ? src : sm;
        const long long ss = (p == 0) ? sstride : smstride;
        cplx* d = (p == P.npass - 1) ? dst : sm;
        const long long ds = (p == P.npass - 1) ? dstride : smstride;
        const int R = P.radix[p];
#define DGPE_PASS(RR, NN)                                                                     \
    case (RR * 8 + NN):                                                                        \
        fft_pass<RR, NN, INV>(P.n, Ns, b, P.nbf, active, s, ss, d, ds, P.tw);                  \
        break;
        switch (R * 8 + P.nb[p]) {
            DGPE_PASS(8, 1)
            DGPE_PASS(4, 1)
            DGPE_PASS(4, 2)
            DGPE_PASS(3, 1)
            DGPE_PASS(3, 2)
            DGPE_PASS(3, 3)
            DGPE_PASS(2, 1)
            DGPE_PASS(2, 2)
            DGPE_PASS(2, 3)
            DGPE_PASS(2, 4)
            DGPE_PASS(5, 1)
            DGPE_PASS(5, 2)
            DGPE_PASS(7, 1)
            DGPE_PASS(7, 2)
            DGPE_PASS(11, 1)
            DGPE_PASS(11, 2)
            DGPE_PASS(13, 1)
            DGPE_PASS(13, 2)
            default: break;
        }
#undef DGPE_PASS
        Ns *= R;
    }
}

}  // namespace dgpe
