// zline.cuh -- the kernels of the contiguous axis z for the specialised line lengths, one WARP per
// z-line (SV section 8a rows a1, a5, a8; BJ:north_star "the R2C density transform fused with the
// |psi|^2 computation on load", "the nonlinear exponential update fused into the inverse-last pass",
// "for the z sweep, the contiguous axis, tiles are ... staged in shared memory so the recursion runs
// along a transposed tile").
//
// A z-line is contiguous in global memory, so a warp reads and writes it with fully coalesced accesses
// and needs no neighbouring lines: every line is an independent job of one warp (of one team of lanes
// for nz <= 256), synchronised with __syncwarp only.  The launchers give every warp its own CTA, so a
// finished line frees its slot at once; 16 (K5) to 28 (K1) warps per SM are in different phases at any
// time, which overlaps the loads, the shared-memory passes, the fp64 arithmetic and the stores without
// block barriers.
//
//   k_z_r2c   (K1)   n = s2 |psi|^2 -> packed nz/2-point FFT -> Hermitian split -> nz/2+1 bins
//   k_z_main  (K5, K8, or both fused) Hermitian merge -> nz/2-point inverse FFT = Phi -> nonlinear
//             exponential -> Crank-Nicolson sweep along z with the chunk of each lane in registers
//
// Shared memory per line:
//   B  FFT buffer, M = nz/2 complex, element idx at idx + (idx >> 3)  (the one pad per 8 elements makes
//      the stride-R writes of the first pass conflict free); the last inverse pass leaves Phi in it as
//      nz plain doubles;
//   A  the psi line, nz complex, LINEAR: it arrives by ONE bulk asynchronous copy (cp.async.bulk, the TMA
//      engine, completion on an mbarrier) and leaves by one bulk store, so no thread issues a global load
//      or store for psi.  Lane l owns the LC unknowns 1 + l LC .. of the line; LC is ODD (17 at nz = 512),
//      so the per-lane walks along the chunks are free of bank conflicts without any padding.
#pragma once
#include "ctfft.cuh"
#include "sweep.cuh"
#include "tma.cuh"
#include <type_traits>

namespace dgpe {

// Lanes per line.  The long lines take a whole warp; for nz/2 = 32 .. 256 (a power of two) a TEAM of
// T = nz/16 lanes owns a line -- then the first FFT pass is one radix-8 butterfly per lane, every lane
// holds 16 psi elements and 17 sweep unknowns exactly as at nz = 512, and a warp works on 32/T lines at
// once with no idle lanes (BJ:configs[0..2]: nz = 64, 128, 256).
__host__ __device__ constexpr int z_team(int nz)
{
    const int m = nz / 2;
    return (m == 32 || m == 64 || m == 128 || m == 256) ? m / 8 : 32;
}

template <int NZ>
struct ZGeom {
    static constexpr int M = NZ / 2;
    static constexpr int T = z_team(NZ);                       // lanes per line
    static constexpr int LPW = 32 / T;                         // lines per warp
    static constexpr int NPER = (NZ + T - 1) / T;              // psi elements per lane (coalesced walks)
    static constexpr int KPER = (M + T - 1) / T;               // spectrum bins per lane
    static constexpr int LC = ((NZ - 2 + T - 1) / T) | 1;      // sweep chunk per lane, odd
    static constexpr int A_ELEMS = NZ;
    static constexpr int B_ELEMS = (M + (M >> 3) + 7) / 8 * 8;
    static_assert(NZ % 2 == 0 && NZ >= 32, "z-line kernels need an even nz >= 32");
};

struct PosPad {
    static __device__ __forceinline__ int at(int idx) { return idx + (idx >> 3); }
};

// shuffles inside a team of W lanes (src = lane index within the team)
template <int W>
__device__ __forceinline__ double shfl_d(double v, int src) { return __shfl_sync(0xffffffffu, v, src, W); }
template <int W>
__device__ __forceinline__ cplx shfl_c(cplx v, int src) { return mk(shfl_d<W>(v.x, src), shfl_d<W>(v.y, src)); }
template <int W>
__device__ __forceinline__ double shfl_ct(double v, int src) { return shfl_d<W>(v, src); }
template <int W>
__device__ __forceinline__ cplx shfl_ct(cplx v, int src) { return shfl_c<W>(v, src); }
__device__ __forceinline__ double ct_zero(double) { return 0.0; }
__device__ __forceinline__ cplx ct_zero(cplx) { return mk(0.0, 0.0); }

// ------------------------------------------------------------------------------------------------
// K1: density + real-to-complex transform along z.  With M = nz/2 the real line is packed as
// z_m = n_{2m} + i n_{2m+1}; Z = DFT_M(z); X_k = (Z_k + conj Z_{M-k})/2 - (i/2) e^{-2 pi i k/nz}
// (Z_k - conj Z_{M-k}), k = 0..M, Z_M := Z_0.   tws[k] = exp(-2 pi i k/nz).
// grid = ceil(nlines / (WARPS LPW)); block = 32*WARPS; dynamic shared memory = WARPS LPW B_ELEMS 16 bytes.
// ------------------------------------------------------------------------------------------------
// DT = cplx: psi is complex (16 bytes per point); DT = double: real-valued psi of the imaginary-time
// fast path (SV section 8f NEXT-2; 8 bytes per point, n = s2 psi^2).
// resident CTAs per SM the register budget of K1 is tuned for: 32 lines (64 registers) pay at nz = 384 (C5: 1.09 -> 0.98 ms);
// at nz = 256, 480, 512 the 28 lines of the compiler's own 68-72 registers are faster (512^3: 0.515 vs 0.553 ms)
template <int NZ>
__host__ __device__ constexpr int k1_min_ctas() { return NZ == 384 ? 32 : 28; }
template <int NZ, int WARPS, typename DT>
__global__ void __launch_bounds__(32 * WARPS, k1_min_ctas<NZ>())
k_z_r2c(const DT* __restrict__ psi, cplx* __restrict__ spec, int nlines, const cplx* __restrict__ tw,
        const cplx* __restrict__ tws, const double* __restrict__ scal)
{
    using G = ZGeom<NZ>;
    constexpr int M = G::M, L = ct::npass(M), TL = G::T, LPW = G::LPW;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int warp = threadIdx.x >> 5, team = (threadIdx.x & 31) / TL, lane = threadIdx.x & (TL - 1);   // lane within the team
    const int line0 = (blockIdx.x * WARPS + warp) * LPW;
    if (line0 >= nlines) return;                        // warps are independent: no block barrier below
    const bool valid = line0 + team < nlines;           // a team past the end works on the last line, stores nothing
    const int line = valid ? line0 + team : nlines - 1;
    cplx* B = reinterpret_cast<cplx*>(smem_raw) + (size_t)(warp * LPW + team) * G::B_ELEMS;
    double* Bd = reinterpret_cast<double*>(B);
    const double s2 = scal[SC_S2];

    constexpr bool RPSI = sizeof(DT) == sizeof(double);
    const DT* p = psi + (long long)line * NZ;
    auto none = [](int) { return mk(0.0, 0.0); };
    auto keep = [&](int idx, cplx v) { B[PosPad::at(idx)] = v; };
    // z_m, m = lane + TL q, is exactly what butterfly `lane` of the first pass reads when that pass has
    // radix M/TL: then each lane loads its pairs (psi_{2m}, psi_{2m+1}) with one 256-bit load -- a warp
    // reads 1 KB contiguous -- and the densities go from registers straight into the pass
    // (also when the first pass has fewer butterflies than the team has lanes -- nz = 480: 30 radix-8
    // butterflies -- the lanes past the last butterfly then sit the first pass out; and with two butterflies
    // per lane, j = lane and lane + TL, when it has more than the team has lanes -- nz = 500, 640, 768: measured
    // at 256 x 256 x nz, complex psi 0.264 -> 0.221 ms (500), 0.234 -> 0.212 (640), but 0.236 -> 0.297 (768);
    // real-valued psi 0.209 -> 0.183, 0.175 -> 0.155, 0.286 -> 0.199)
    using P0 = CtPass<M, 0, false, false, TL>;
    constexpr bool FIRST_IN_REGS = P0::Ns == 1 && (P0::NB == 1 || (P0::NB == 2 && (RPSI || NZ <= 640)));
    if constexpr (FIRST_IN_REGS) {
        constexpr int NB0 = P0::NBUT, NBU = P0::NB;      // butterfly j reads z_m, m = j + NB0 q
        P0 p0;
        if constexpr (RPSI) {
            // the pair (psi_{2m}, psi_{2m+1}) is one 128-bit load: a warp reads 512 bytes contiguous
            cplx w[NBU][P0::R];
#pragma unroll
            for (int u = 0; u < NBU; ++u)
#pragma unroll
                for (int q = 0; q < P0::R; ++q) {
                    const int j = lane + u * TL;
                    w[u][q] = (P0::EXACT || j < NB0) ? ld_stream(reinterpret_cast<const cplx*>(p + 2 * (j + NB0 * q))) : mk(0.0, 0.0);
                }
#pragma unroll
            for (int u = 0; u < NBU; ++u)
#pragma unroll
                for (int q = 0; q < P0::R; ++q) p0.v[u][q] = mk(s2 * (w[u][q].x * w[u][q].x), s2 * (w[u][q].y * w[u][q].y));
        } else {
            double4 w[NBU][P0::R];
#pragma unroll
            for (int u = 0; u < NBU; ++u)
#pragma unroll
                for (int q = 0; q < P0::R; ++q) {
                    const int j = lane + u * TL;
                    const double* src = reinterpret_cast<const double*>(p + 2 * (j + NB0 * q));
                    w[u][q] = make_double4(0.0, 0.0, 0.0, 0.0);
                    if (P0::EXACT || j < NB0)
                        asm volatile("ld.global.cs.v4.f64 {%0, %1, %2, %3}, [%4];\n"
                                     : "=d"(w[u][q].x), "=d"(w[u][q].y), "=d"(w[u][q].z), "=d"(w[u][q].w)
                                     : "l"(src));
                }
#pragma unroll
            for (int u = 0; u < NBU; ++u)
#pragma unroll
                for (int q = 0; q < P0::R; ++q)
                    p0.v[u][q] = mk(s2 * (w[u][q].x * w[u][q].x + w[u][q].y * w[u][q].y),
                                    s2 * (w[u][q].z * w[u][q].z + w[u][q].w * w[u][q].w));
        }
        p0.bfly(lane);
        if constexpr (P0::LAST) {
            p0.scatter(lane, keep);
        } else {
            p0.scatter(lane, keep);
            __syncwarp();
            ct_fft_range<M, false, false, TL, SyncWarp, PosPad, 1, L, false>(B, lane, true, tw, none, keep);
        }
    } else {
        DT a[G::NPER];
#pragma unroll
        for (int i = 0; i < G::NPER; ++i) {
            const int e = TL * i + lane;
            a[i] = (NZ % TL == 0 || e < NZ) ? ld_stream(p + e) : ct_zero(DT());
        }
#pragma unroll
        for (int i = 0; i < G::NPER; ++i) {
            const int e = TL * i + lane, m = e >> 1;
            if (NZ % TL == 0 || e < NZ) Bd[2 * PosPad::at(m) + (e & 1)] = s2 * cabs2(a[i]);
        }
        __syncwarp();
        ct_fft_range<M, false, false, TL, SyncWarp, PosPad, 0, L, false>(B, lane, true, tw, none, keep);
    }
    __syncwarp();

    cplx* out = spec + (long long)line * (M + 1);
    auto split = [&](int k) {
        const int k1 = (k == M) ? 0 : k, k2 = (k == 0) ? 0 : M - k;
        const cplx zk = B[PosPad::at(k1)];
        const cplx zm = cconj(B[PosPad::at(k2)]);
        const cplx w = __ldg(&tws[k]);
        const cplx s = cadd(zk, zm), d = csub(zk, zm);
        const cplx wd = cmul(w, d);
        if (valid) st_stream(out + k, mk(0.5 * (s.x + wd.y), 0.5 * (s.y - wd.x)));     // s/2 - (i/2) w d
    };
#pragma unroll
    for (int t = 0; t < G::KPER; ++t)
        if (M % TL == 0 || lane + TL * t < M) split(lane + TL * t);
    if (lane == 0) split(M);
}

// ------------------------------------------------------------------------------------------------
// K5 / K8: everything that happens to one z-line of psi between two strided passes.
//   SPEC = ZS_NONE    only the sweep (dgpe_sweep along z)
//   SPEC = ZS_IMAG    C2R + psi <- exp(-dt H) s1 psi              (BJ:north_star (b), imaginary time)
//   SPEC = ZS_REAL    C2R + psi <- (cos(dt H) - i sin(dt H)) psi  (real time)
//   SPEC = ZS_PHI     C2R, Phi written to phi_out (dgpe_dipolar); psi untouched
//   SWEEP             followed by the Crank-Nicolson sweep along z of the same line while it is still
//                     in shared memory (the three 1-D Cayley operators commute, so the step may run
//                     its sweeps in the order z, x, y: DESIGN.md R#26) -- this removes one full
//                     read+write pass over psi (32N bytes) from the step.
// C2R: from the half-spectrum X_0..X_M of the line, Z_k = (X_k + conj X_{M-k}) + i e^{+2 pi i k/nz}
// (X_k - conj X_{M-k}), k = 0..M-1; z = IDFT_M(Z) (the 1/N is already in K3); Phi_{2m} = Re z_m,
// Phi_{2m+1} = Im z_m.   H = V + g n + gdd Phi, n = s2 |psi|^2, V = (vx[i] + vy[j] + vz[k])/2.
// Sweep: as sweep.cuh; lane l owns the unknowns 1 + l LC .. and keeps them in registers through the
// forward elimination, the back substitution and the fix-up; the chunk outflows travel by shuffles.
// grid = ceil(nlines / (WARPS LPW)); block = 32*WARPS; dynamic smem = WARPS LPW (A_ELEMS sizeof(DT) + B_ELEMS 16) bytes.
// ------------------------------------------------------------------------------------------------
enum { ZS_NONE = 0, ZS_IMAG = 1, ZS_REAL = 2, ZS_PHI = 3 };

struct ZMainArgs {
    int nlines, ny;
    double dt, g, gdd;
    double dz, lam2;       // z_k = (k - nz/2) dz, V_z = lambda^2 z_k^2 / 2 (evaluated in the kernel, no table walk)
    const double *vx, *vy;
    const double* scal;
    const cplx* tw;        // exp(-2 pi i j/M)
    const cplx* tws;       // exp(-2 pi i k/nz)
    double* phi_out;       // ZS_PHI
    int pf_lines;          // L2 prefetch distance in lines (= lines resident on the GPU at a time); 0 = off
};

// one bulk asynchronous copy global -> shared (TMA engine), completion counted on an mbarrier
__device__ __forceinline__ void bulk_load(void* smem_dst, const void* gsrc, unsigned bytes, unsigned long long* bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];\n" ::"r"(
                     smem_addr(smem_dst)),
                 "l"(gsrc), "r"(bytes), "r"(smem_addr(bar))
                 : "memory");
}
// one bulk asynchronous copy shared -> global, tracked by the issuing thread's bulk async-groups
__device__ __forceinline__ void bulk_store(void* gdst, const void* smem_src, unsigned bytes)
{
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;\n" ::"l"(gdst), "r"(smem_addr(smem_src)),
                 "r"(bytes)
                 : "memory");
}

// DT = cplx, or double for the real-valued psi of the imaginary-time fast path (CT = double, SPEC != ZS_REAL):
// the line buffer A then holds nz doubles, and every quantity of the sweep is one double instead of two.
template <int NZ, typename CT, typename DT, int SPEC, bool SWEEP, bool CONSTTAB, int WARPS, int MINB>
__global__ void __launch_bounds__(32 * WARPS, MINB)
k_z_main(DT* __restrict__ psi, const cplx* __restrict__ spec, ZMainArgs Z, SweepTables<CT> T,
         const CT* __restrict__ ptab, const __grid_constant__ ChunkTabs<CT, ZGeom<NZ>::LC> P)
{
    using G = ZGeom<NZ>;
    constexpr int M = G::M, L = ct::npass(M), LC = G::LC, TL = G::T, LPW = G::LPW;
    constexpr bool USE_A = (SPEC != ZS_PHI);
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ __align__(8) unsigned long long bars[WARPS * LPW];
    const int warp = threadIdx.x >> 5, team = (threadIdx.x & 31) / TL, lane = threadIdx.x & (TL - 1);   // lane within the team
    const int line0 = (blockIdx.x * WARPS + warp) * LPW;
    if (line0 >= Z.nlines) return;                      // warps are independent: no block barrier below
    const bool valid = line0 + team < Z.nlines;         // a team past the end works on the last line, stores nothing
    const int line = valid ? line0 + team : Z.nlines - 1;
    const int slot = warp * LPW + team;
    static_assert(sizeof(DT) == sizeof(cplx) || (sizeof(CT) == sizeof(double) && SPEC != ZS_REAL),
                  "real-valued psi: imaginary time only");
    constexpr unsigned A_BYTES = USE_A ? G::A_ELEMS * (unsigned)sizeof(DT) : 0u;      // a multiple of 16 (nz even)
    constexpr unsigned PER_LINE = A_BYTES + (SPEC != ZS_NONE ? G::B_ELEMS * (unsigned)sizeof(cplx) : 0u);
    DT* A = reinterpret_cast<DT*>(smem_raw + (size_t)slot * PER_LINE);
    cplx* B = reinterpret_cast<cplx*>(smem_raw + (size_t)slot * PER_LINE + A_BYTES);
    DT* p = psi + (long long)line * NZ;

    // ---- the psi line: one bulk copy, in flight while the spectrum is loaded, merged and transformed ----
    if constexpr (USE_A) {
        if (lane == 0) {
            mbar_init(&bars[slot], 1);
            mbar_fence_init();
            mbar_expect_tx(&bars[slot], A_BYTES);
            bulk_load(A, p, A_BYTES, &bars[slot]);
        }
    }
    // ---- L2 prefetch for the warp that will run one residency later ----
    if (Z.pf_lines > 0 && line + Z.pf_lines < Z.nlines) {
        const char* pp = reinterpret_cast<const char*>(psi + (long long)(line + Z.pf_lines) * NZ);
        if constexpr (USE_A) {
            for (int o = 128 * lane; o < (int)A_BYTES; o += 128 * TL) prefetch_l2(pp + o);
        }
        if constexpr (SPEC != ZS_NONE) {
            const char* ps = reinterpret_cast<const char*>(spec + (long long)(line + Z.pf_lines) * (M + 1));
            for (int o = 128 * lane; o < (M + 1) * 16; o += 128 * TL) prefetch_l2(ps + o);
        }
    }

    if constexpr (SPEC != ZS_NONE) {
        // ---- Hermitian merge straight from global memory ----
        // Z_k, k = lane + TL t, is exactly what butterfly `lane` of the first inverse pass reads when that
        // pass has radix M/TL: then the merged values go from registers straight into the pass
        // (or fewer butterflies than lanes: the bins are then dealt out with the butterfly count as the stride)
        using P0 = CtPass<M, 0, true, false, TL>;
        // (one butterfly per lane only: with two, the 2 x 2 R merged bins in registers slow this kernel down --
        // measured at nz = 500, 640, 768)
        constexpr bool FIRST_IN_REGS = P0::NB == 1 && P0::Ns == 1;
        // lane's bins: t = u R + q -> k = (lane + u TL) + NBUT q (butterfly j = lane + u TL of the first pass), else k = lane + TL t
        constexpr int KCNT = FIRST_IN_REGS ? P0::NB * P0::R : G::KPER;
        auto bin = [&](int t) {
            if constexpr (FIRST_IN_REGS) return min(lane + (t / P0::R) * TL + P0::NBUT * (t % P0::R), M - 1);
            else return min(lane + TL * t, M - 1);                // (bins past M-1: loaded twice, never stored)
        };
        const cplx* in = spec + (long long)line * (M + 1);
        cplx xa[KCNT], xb[KCNT];
#pragma unroll
        for (int t = 0; t < KCNT; ++t) {
            const int k = bin(t);
            xa[t] = ld_stream(in + k);
            xb[t] = ld_stream(in + (M - k));
        }
#pragma unroll
        for (int t = 0; t < KCNT; ++t) {
            const int k = bin(t);
            const cplx w = cconj(__ldg(&Z.tws[k]));               // e^{+2 pi i k/nz}
            const cplx cb = cconj(xb[t]);
            const cplx s = cadd(xa[t], cb), d = csub(xa[t], cb);
            const cplx wd = cmul(w, d);
            xa[t] = mk(s.x - wd.y, s.y + wd.x);                   // Z_k = s + i w d
        }
        // the last pass leaves z_m = Phi_{2m} + i Phi_{2m+1} at B[m], unpadded: Phi as nz plain doubles
        auto keep_phi = [&](int m, cplx phi) {
            if constexpr (SPEC == ZS_PHI) { if (valid) reinterpret_cast<double2*>(Z.phi_out + (long long)line * NZ)[m] = phi; }
            else B[m] = phi;
        };
        auto none = [](int) { return mk(0.0, 0.0); };
        if constexpr (FIRST_IN_REGS) {
            P0 p0;
#pragma unroll
            for (int u = 0; u < P0::NB; ++u)
#pragma unroll
                for (int q = 0; q < P0::R; ++q) p0.v[u][q] = xa[u * P0::R + q];
            p0.bfly(lane);
            if constexpr (P0::LAST) {
                p0.scatter(lane, keep_phi);
            } else {
                p0.scatter(lane, [&](int idx, cplx val) { B[PosPad::at(idx)] = val; });
                __syncwarp();
                ct_fft_range<M, true, false, TL, SyncWarp, PosPad, 1, L, false>(B, lane, true, Z.tw, none, keep_phi);
            }
        } else {
#pragma unroll
            for (int t = 0; t < G::KPER; ++t)
                if (M % TL == 0 || lane + TL * t < M) B[PosPad::at(lane + TL * t)] = xa[t];
            __syncwarp();
            ct_fft_range<M, true, false, TL, SyncWarp, PosPad, 0, L, false>(B, lane, true, Z.tw, none, keep_phi);
        }
    }
    __syncwarp();
    if constexpr (!USE_A) return;
    mbar_wait(&bars[slot], 0u);                          // the psi line has landed

    // ---- psi_e after the nonlinear / potential exponential (or as it stands: ZS_NONE) ----
    const double* Bd = reinterpret_cast<const double*>(B);
    double vxy = 0.0, s2 = 1.0, s1 = 1.0;
    if constexpr (SPEC != ZS_NONE) {
        const int i = line / Z.ny, j = line - i * Z.ny;
        vxy = __ldg(&Z.vx[i]) + __ldg(&Z.vy[j]);
        s2 = Z.scal[SC_S2];
        s1 = Z.scal[SC_S1];
    }
    // PRECISE = false: the branch-free sincos_fast; it is exact to 2e-16 below SINCOS_FAST_LIMIT, and `big` records
    // an argument at or beyond it (or a NaN), for which the caller evaluates the point again with PRECISE = true
    // (the library's sincos with its exact reduction) -- never taken for the phases of a physical state
    bool big = false;
    auto upd_as = [&](int e, auto precise) -> DT {
        DT a = A[e];
        if constexpr (SPEC == ZS_IMAG || SPEC == ZS_REAL) {
            const double z = (double)(e - NZ / 2) * Z.dz;          // R#6
            const double vz = Z.lam2 * z * z;
            const double dens = s2 * cabs2(a);
            const double H = 0.5 * (vxy + vz) + Z.g * dens + Z.gdd * Bd[e];
            if constexpr (SPEC == ZS_IMAG) {
                const double f = exp(-Z.dt * H) * s1;
                a = coef_mul(f, a);
            } else {
                const double th = Z.dt * H;
                double sn, cs;
                if constexpr (decltype(precise)::value) {
                    sincos(th, &sn, &cs);
                } else {
                    sincos_fast(th, &sn, &cs);
                    big |= !(fabs(th) < SINCOS_FAST_LIMIT);
                }
                a = mk(cs * a.x + sn * a.y, cs * a.y - sn * a.x);
            }
        }
        return a;
    };
    auto upd = [&](int e) -> DT { return upd_as(e, std::false_type()); };

    const int s = 1 + lane * LC;
    const int cnt = min(LC, NZ - 1 - s);                  // unknowns of this lane's chunk (<= 0: idle lane)
    if constexpr (SWEEP) {
        const int Gn = T.G;
        // table base of this lane (CONSTTAB = false): away from the left wall the elimination factors have
        // converged, so the interior chunks share one set of entries (T.gU) -- one broadcast address
        const int sT = (lane >= T.gU && lane < Gn - 1) ? 1 + T.gU * LC : s;
        // CONSTTAB: the Thomas factors of chunk 0 and of the converged chunk as ONE compact table of 8 LC entries
        // (ptab, built on the host: [inv, cc, F, Gm] of chunk 0, then of the converged chunk; F of chunk 0 multiplies a
        // zero inflow), read through L1 with the lane-0 / other-lanes choice in the address: one load per factor, two
        // addresses per warp.  (As kernel parameters every factor cost three LDC per double -- one for chunk 0, two
        // predicated ones for the converged chunk -- and the constant-load unit was the busiest pipe of the real-time
        // kernel: 60 % in ncu.  A copy in shared memory costs the 16th resident line at nz = 256 and 512.)
        // Real-valued psi (every quantity one double, half the factors): there the kernel parameters stay faster
        // (measured at 512^3: 0.709 vs 0.738 ms).
        constexpr bool PARAMTAB = CONSTTAB && sizeof(DT) == sizeof(double);
        const CT* tb = ptab + (lane == 0 ? 0 : 4 * LC);
        const bool l0 = lane == 0;
        auto t_inv = [&](int i) {
            if constexpr (PARAMTAB) return l0 ? P.inv0[i] : P.invU[i];
            else if constexpr (CONSTTAB) return __ldg(&tb[i]);
            else return __ldg(&T.inv[sT + i]);
        };
        auto t_cc = [&](int i) {
            if constexpr (PARAMTAB) return l0 ? P.cc0[i] : P.ccU[i];
            else if constexpr (CONSTTAB) return __ldg(&tb[LC + i]);
            else return __ldg(&T.cc[sT + i]);
        };
        auto t_F = [&](int i) {
            if constexpr (PARAMTAB) return P.fU[i];
            else if constexpr (CONSTTAB) return __ldg(&tb[2 * LC + i]);
            else return __ldg(&T.F[sT + i]);
        };
        auto t_Gm = [&](int i) {
            if constexpr (PARAMTAB) return l0 ? P.gm0[i] : P.gmU[i];
            else if constexpr (CONSTTAB) return __ldg(&tb[3 * LC + i]);
            else return __ldg(&T.Gm[sT + i]);
        };

        // ---- A: nonlinear update on the fly + local forward elimination with zero inflow; the end nodes
        //      of the line are read as zero (R#7, R#8).
        // (branch-free: every lane evaluates its LC updates on clamped indices and masks the ones past its
        // chunk or on an end node, so the exponentials of one lane interleave; the two halo values come
        // from the neighbouring lanes by shuffles -- every lane left of an active lane owns a full chunk)
        const DT zero = ct_zero(DT());
        DT pv[LC + 2];
#pragma unroll
        for (int i = 1; i <= LC; ++i) {
            const int j = s - 1 + i;
            const DT v = upd(min(j, NZ - 1));
            pv[i] = el_sel(j <= NZ - 2, v, zero);
        }
        if constexpr (SPEC == ZS_REAL) {
            if (big) {                                   // rare: a phase beyond the fast reduction's range
#pragma unroll 1
                for (int i = 1; i <= LC; ++i) {
                    const int j = s - 1 + i;
                    const DT v = upd_as(min(j, NZ - 1), std::true_type());
                    const DT w = el_sel(j <= NZ - 2, v, zero);
                    // pv is a register array: select the entry without dynamic indexing
#pragma unroll
                    for (int u = 1; u <= LC; ++u) pv[u] = el_sel(u == i, w, pv[u]);
                }
            }
        }
        {
            const DT up = shfl_ct<TL>(pv[LC], (lane + TL - 1) & (TL - 1)), dn = shfl_ct<TL>(pv[1], (lane + 1) & (TL - 1));
            pv[0] = (lane == 0) ? zero : up;
            pv[LC + 1] = (lane == TL - 1) ? zero : dn;
        }
        DT ev[LC];
        DT e = zero;
#pragma unroll
        for (int i = 0; i < LC; ++i) {
            // inv_j (d_j + r e_{j-1}) = inv_j d_j + (-c_j) e_{j-1}: one dependent fma per unknown
            const DT d = cn_rhs(T.r, T.omr2, pv[i], pv[i + 1], pv[i + 2]);
            const DT en = coef_fma(coef_neg(t_cc(i)), e, coef_mul(t_inv(i), d));
            e = el_sel(i < cnt, en, e);
            ev[i] = e;
        }
        // ---- B: forward inflow by a look-back over the lanes to the left ----
        const CT Ag = (lane < Gn) ? __ldg(&T.Ach[lane]) : ct_zero(CT());
        const CT Bg = (lane < Gn) ? __ldg(&T.Bch[lane]) : ct_zero(CT());
        DT ein = zero;
        for (int d = T.Kf; d >= 1; --d) {
            const int h = lane - d;
            const DT Eh = shfl_ct<TL>(e, h & (TL - 1));
            const CT Ah = shfl_ct<TL>(Ag, h & (TL - 1));
            if (h >= 0) ein = coef_fma(Ah, ein, Eh);
        }
        // ---- C: local back substitution with zero inflow ----
        DT x = zero;
#pragma unroll
        for (int i = LC - 1; i >= 0; --i) {
            if (i < cnt) {
                const DT ee = coef_fma(t_F(i), ein, ev[i]);
                x = coef_fma(coef_neg(t_cc(i)), x, ee);
                ev[i] = x;
            }
        }
        // ---- D: backward inflow from the lanes to the right ----
        DT xin = zero;
        for (int d = T.Kb; d >= 1; --d) {
            const int h = lane + d;
            const DT Xh = shfl_ct<TL>(x, h & (TL - 1));
            const CT Bh = shfl_ct<TL>(Bg, h & (TL - 1));
            if (h < Gn) xin = coef_fma(Bh, xin, Xh);
        }
        __syncwarp();                                    // every lane has read its halo from the line buffer
        // ---- E: final values back into the line buffer; Dirichlet end nodes are exact zeros ----
#pragma unroll
        for (int i = 0; i < LC; ++i)
            if (i < cnt) A[s + i] = coef_fma(t_Gm(i), xin, ev[i]);
        if (lane == 0) A[0] = zero;
        if (lane == TL - 1) A[NZ - 1] = zero;
    } else {
        // nonlinear update only (dgpe_nonlinear): every point of the line, end nodes included
        // (dgpe_nonlinear, not the step: same fast sincos, the fallback decided point by point)
        auto upd_checked = [&](int e) -> DT {
            big = false;
            DT v = upd(e);
            if (big) v = upd_as(e, std::true_type());
            return v;
        };
#pragma unroll
        for (int i = 0; i < LC; ++i)
            if (i < cnt) A[s + i] = upd_checked(s + i);
        if (lane == 0) A[0] = upd_checked(0);
        if (lane == TL - 1) A[NZ - 1] = upd_checked(NZ - 1);
    }

    // ---- the line goes back by one bulk store ----
    fence_proxy_async();                                 // my writes -> visible to the async proxy
    __syncwarp();
    if (lane == 0 && valid) {
        bulk_store(p, A, A_BYTES);
        tma_store_commit();
        tma_store_wait_read<0>();                        // shared memory must outlive the copy
    }
}

}  // namespace dgpe
