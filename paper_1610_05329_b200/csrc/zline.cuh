// zline.cuh -- the kernels of the contiguous axis z for the specialised line lengths, one WARP per
// z-line (SV section 8a rows a1, a5, a8; BJ:north_star "the R2C density transform fused with the
// |psi|^2 computation on load", "the nonlinear exponential update fused into the inverse-last pass",
// "for the z sweep, the contiguous axis, tiles are ... staged in shared memory so the recursion runs
// along a transposed tile").
//
// A z-line is contiguous in global memory, so a warp reads and writes it with fully coalesced 512-byte
// accesses and needs no neighbouring lines: every line is an independent job of one warp, synchronised
// with __syncwarp only.  Many warps per SM (16 at 512^3) are in different phases at any time, which
// overlaps the loads, the shared-memory passes, the fp64 arithmetic and the stores without block
// barriers.
//
//   k_z_r2c   (K1)   n = s2 |psi|^2 -> packed nz/2-point FFT -> Hermitian split -> nz/2+1 bins
//   k_z_main  (K5, K8, or both fused) Hermitian merge -> nz/2-point inverse FFT = Phi -> nonlinear
//             exponential -> Crank-Nicolson sweep along z with the chunk of each lane in registers
//
// Shared memory per warp:
//   B  FFT buffer, M = nz/2 complex, element idx at idx + (idx >> 3)  (the one pad per 8 elements makes
//      the stride-R writes of the first pass conflict free);
//   A  the psi line, even and odd elements in two padded halves (PosLine): the coalesced walks along the
//      line, the pair walk of the nonlinear update and the per-lane walks along a sweep chunk are all
//      conflict free.
#pragma once
#include "ctfft.cuh"
#include "sweep.cuh"

namespace dgpe {

template <int NZ>
struct ZGeom {
    static constexpr int M = NZ / 2;
    static constexpr int NPER = NZ / 32;                 // psi elements per lane
    static constexpr int LC = (NZ - 2 + 31) / 32;        // sweep chunk per lane
    static constexpr int HALF = ((M + (M >> 3) + 7) / 8) * 8 + 4;      // offset of the odd half, = 4 mod 8
    static constexpr int A_ELEMS = (HALF + M + (M >> 3) + 7) / 8 * 8;
    static constexpr int B_ELEMS = (M + (M >> 3) + 7) / 8 * 8;
    static_assert(NZ % 64 == 0, "z-line kernels need nz to be a multiple of 64");
    static_assert(LC % 2 == 0, "the chunk walk is conflict free only for an even chunk length");
};

struct PosPad {
    static __device__ __forceinline__ int at(int idx) { return idx + (idx >> 3); }
};

// Line buffer A: element e = 2m + t lives at t*HALF + m + (m >> 3).  Three access patterns are all
// free of bank conflicts (16-byte elements: the 8 lanes of a quarter-warp must hit 8 different
// positions mod 8):  the coalesced walk (lane <-> e), 4 even and 4 odd elements per quarter-warp, the
// halves 4 banks apart;  the pair walk of the nonlinear update (lane <-> m);  the chunk walk of the
// sweep (lane <-> e = 1 + LC lane + i, LC even: m advances by LC/2 per lane, the pad makes the stride odd
// for LC = 16).
template <int NZ>
struct PosLine {
    static __device__ __forceinline__ int at(int e)
    {
        const int m = e >> 1;
        return (e & 1) * ZGeom<NZ>::HALF + m + (m >> 3);
    }
};

__device__ __forceinline__ double shfl_d(double v, int src) { return __shfl_sync(0xffffffffu, v, src); }
__device__ __forceinline__ cplx shfl_c(cplx v, int src) { return mk(shfl_d(v.x, src), shfl_d(v.y, src)); }
__device__ __forceinline__ double shfl_ct(double v, int src) { return shfl_d(v, src); }
__device__ __forceinline__ cplx shfl_ct(cplx v, int src) { return shfl_c(v, src); }
__device__ __forceinline__ double ct_zero(double) { return 0.0; }
__device__ __forceinline__ cplx ct_zero(cplx) { return mk(0.0, 0.0); }

// ------------------------------------------------------------------------------------------------
// K1: density + real-to-complex transform along z.  With M = nz/2 the real line is packed as
// z_m = n_{2m} + i n_{2m+1}; Z = DFT_M(z); X_k = (Z_k + conj Z_{M-k})/2 - (i/2) e^{-2 pi i k/nz}
// (Z_k - conj Z_{M-k}), k = 0..M, Z_M := Z_0.   tws[k] = exp(-2 pi i k/nz).
// grid = ceil(nlines / WARPS); block = 32*WARPS; dynamic shared memory = WARPS * B_ELEMS * 16 bytes.
// ------------------------------------------------------------------------------------------------
template <int NZ, int WARPS>
__global__ void __launch_bounds__(32 * WARPS)
k_z_r2c(const cplx* __restrict__ psi, cplx* __restrict__ spec, int nlines, const cplx* __restrict__ tw,
        const cplx* __restrict__ tws, const double* __restrict__ scal)
{
    using G = ZGeom<NZ>;
    constexpr int M = G::M, L = ct::npass(M);
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int line = blockIdx.x * WARPS + warp;
    if (line >= nlines) return;                         // warps are independent: no block barrier below
    cplx* B = reinterpret_cast<cplx*>(smem_raw) + (size_t)warp * G::B_ELEMS;
    double* Bd = reinterpret_cast<double*>(B);
    const double s2 = scal[SC_S2];

    const cplx* p = psi + (long long)line * NZ;
    cplx a[G::NPER];
#pragma unroll
    for (int i = 0; i < G::NPER; ++i) a[i] = ld_stream(p + 32 * i + lane);
#pragma unroll
    for (int i = 0; i < G::NPER; ++i) {
        const int e = 32 * i + lane, m = e >> 1;
        Bd[2 * PosPad::at(m) + (e & 1)] = s2 * cabs2(a[i]);
    }
    __syncwarp();

    auto none = [](int) { return mk(0.0, 0.0); };
    ct_fft_range<M, false, false, 32, SyncWarp, PosPad, 0, L, false>(
        B, lane, true, tw, none, [&](int idx, cplx v) { B[PosPad::at(idx)] = v; });
    __syncwarp();

    cplx* out = spec + (long long)line * (M + 1);
    auto split = [&](int k) {
        const int k1 = (k == M) ? 0 : k, k2 = (k == 0) ? 0 : M - k;
        const cplx zk = B[PosPad::at(k1)];
        const cplx zm = cconj(B[PosPad::at(k2)]);
        const cplx w = __ldg(&tws[k]);
        const cplx s = cadd(zk, zm), d = csub(zk, zm);
        const cplx wd = cmul(w, d);
        st_stream(out + k, mk(0.5 * (s.x + wd.y), 0.5 * (s.y - wd.x)));     // s/2 - (i/2) w d
    };
#pragma unroll
    for (int t = 0; t < M / 32; ++t) split(lane + 32 * t);
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
// grid = ceil(nlines / WARPS); block = 32*WARPS; dynamic smem = WARPS*(A_ELEMS + B_ELEMS)*16 bytes.
// ------------------------------------------------------------------------------------------------
enum { ZS_NONE = 0, ZS_IMAG = 1, ZS_REAL = 2, ZS_PHI = 3 };

struct ZMainArgs {
    int nlines, ny;
    double dt, g, gdd;
    const double *vx, *vy, *vz;
    const double* scal;
    const cplx* tw;        // exp(-2 pi i j/M)
    const cplx* tws;       // exp(-2 pi i k/nz)
    double* phi_out;       // ZS_PHI
    int pf_lines;          // L2 prefetch distance in lines (= lines resident on the GPU at a time); 0 = off
};

template <int NZ, typename CT, int SPEC, bool SWEEP, bool CONSTTAB, int WARPS, int MINB>
__global__ void __launch_bounds__(32 * WARPS, MINB)
k_z_main(cplx* __restrict__ psi, const cplx* __restrict__ spec, ZMainArgs Z, SweepTables<CT> T,
         const __grid_constant__ ChunkTabs<CT, ZGeom<NZ>::LC> P)
{
    using G = ZGeom<NZ>;
    using PL = PosLine<NZ>;
    constexpr int M = G::M, L = ct::npass(M), LC = G::LC;
    constexpr bool USE_A = (SPEC != ZS_PHI);
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int line = blockIdx.x * WARPS + warp;
    if (line >= Z.nlines) return;                       // warps are independent: no block barrier below
    constexpr int PER_WARP = (USE_A ? G::A_ELEMS : 0) + (SPEC != ZS_NONE ? G::B_ELEMS : 0);
    cplx* A = reinterpret_cast<cplx*>(smem_raw) + (size_t)warp * PER_WARP;
    cplx* B = A + (USE_A ? G::A_ELEMS : 0);
    cplx* p = psi + (long long)line * NZ;

    // ---- stage the psi line and merge the half-spectrum; the global loads of both are issued before
    //      anything waits on them (psi in two batches to bound the registers in flight) ----
    // ---- L2 prefetch for the warp that will run one residency later ----
    if (Z.pf_lines > 0 && line + Z.pf_lines < Z.nlines) {
        const char* pp = reinterpret_cast<const char*>(psi + (long long)(line + Z.pf_lines) * NZ);
        if constexpr (USE_A) {
#pragma unroll
            for (int i = 0; i < (NZ * 16) / (128 * 32); ++i) prefetch_l2(pp + 128 * (lane + 32 * i));
            if ((NZ * 16) % (128 * 32) != 0 && lane < ((NZ * 16) % (128 * 32)) / 128)
                prefetch_l2(pp + 128 * (lane + 32 * ((NZ * 16) / (128 * 32))));
        }
        if constexpr (SPEC != ZS_NONE) {
            const char* ps = reinterpret_cast<const char*>(spec + (long long)(line + Z.pf_lines) * (M + 1));
            for (int o = 128 * lane; o < (M + 1) * 16; o += 128 * 32) prefetch_l2(ps + o);
        }
    }
    constexpr int HB = G::NPER / 2;
    cplx a[HB];
    // Z_k, k = lane + 32 t, is exactly what butterfly `lane` of the first inverse pass reads when that pass
    // has radix M/32: then the merged values go from registers straight into the pass
    constexpr bool FIRST_IN_REGS = (SPEC != ZS_NONE) && (ct::radix_at(M, 0, false) == M / 32);
    cplx xa[SPEC != ZS_NONE ? M / 32 : 1];
    if constexpr (USE_A) {
#pragma unroll
        for (int i = 0; i < HB; ++i) a[i] = ld_stream(p + 32 * i + lane);
    }
    if constexpr (SPEC != ZS_NONE) {
        // Hermitian merge straight from global memory into the FFT buffer
        const cplx* in = spec + (long long)line * (M + 1);
        cplx xb[M / 32];
#pragma unroll
        for (int t = 0; t < M / 32; ++t) {
            const int k = lane + 32 * t;
            xa[t] = ld_stream(in + k);
            xb[t] = ld_stream(in + (M - k));
        }
        if constexpr (USE_A) {
#pragma unroll
            for (int i = 0; i < HB; ++i) A[PL::at(32 * i + lane)] = a[i];
#pragma unroll
            for (int i = 0; i < HB; ++i) a[i] = ld_stream(p + 32 * (HB + i) + lane);
        }
#pragma unroll
        for (int t = 0; t < M / 32; ++t) {
            const int k = lane + 32 * t;
            const cplx w = cconj(__ldg(&Z.tws[k]));               // e^{+2 pi i k/nz}
            const cplx cb = cconj(xb[t]);
            const cplx s = cadd(xa[t], cb), d = csub(xa[t], cb);
            const cplx wd = cmul(w, d);
            xa[t] = mk(s.x - wd.y, s.y + wd.x);                   // Z_k = s + i w d
        }
        if constexpr (!FIRST_IN_REGS) {
#pragma unroll
            for (int t = 0; t < M / 32; ++t) B[PosPad::at(lane + 32 * t)] = xa[t];
        }
        if constexpr (USE_A) {
#pragma unroll
            for (int i = 0; i < HB; ++i) A[PL::at(32 * (HB + i) + lane)] = a[i];
        }
    } else {
#pragma unroll
        for (int i = 0; i < HB; ++i) A[PL::at(32 * i + lane)] = a[i];
#pragma unroll
        for (int i = 0; i < HB; ++i) a[i] = ld_stream(p + 32 * (HB + i) + lane);
#pragma unroll
        for (int i = 0; i < HB; ++i) A[PL::at(32 * (HB + i) + lane)] = a[i];
    }
    __syncwarp();

    if constexpr (SPEC != ZS_NONE) {
        const int i = line / Z.ny, j = line - i * Z.ny;
        const double vxy = __ldg(&Z.vx[i]) + __ldg(&Z.vy[j]);
        const double s2 = Z.scal[SC_S2], s1 = Z.scal[SC_S1];
        auto none = [](int) { return mk(0.0, 0.0); };
        auto nonlin = [&](int m, cplx phi) {
            if constexpr (SPEC == ZS_PHI) {
                reinterpret_cast<double2*>(Z.phi_out + (long long)line * NZ)[m] = phi;
            } else {
                const double2 vz = __ldg(reinterpret_cast<const double2*>(Z.vz) + m);
                const double vzz[2] = {vz.x, vz.y}, ph[2] = {phi.x, phi.y};
#pragma unroll
                for (int t = 0; t < 2; ++t) {
                    const int pos = PL::at(2 * m + t);
                    cplx a = A[pos];
                    const double dens = s2 * cabs2(a);
                    const double H = 0.5 * (vxy + vzz[t]) + Z.g * dens + Z.gdd * ph[t];
                    if constexpr (SPEC == ZS_IMAG) {
                        const double f = exp(-Z.dt * H) * s1;
                        a = mk(f * a.x, f * a.y);
                    } else {
                        double sn, cs;
                        sincos(Z.dt * H, &sn, &cs);
                        a = mk(cs * a.x + sn * a.y, cs * a.y - sn * a.x);
                    }
                    A[pos] = a;
                }
            }
        };
        if constexpr (FIRST_IN_REGS) {
            using P0 = CtPass<M, 0, true, false, 32>;
            static_assert(P0::NB == 1 && P0::R == M / 32 && P0::Ns == 1, "first pass must be one butterfly per lane");
            P0 p0;
#pragma unroll
            for (int q = 0; q < P0::R; ++q) p0.v[0][q] = xa[q];
            p0.bfly(lane);
            if constexpr (P0::LAST) {
                p0.scatter(lane, nonlin);
            } else {
                p0.scatter(lane, [&](int idx, cplx val) { B[PosPad::at(idx)] = val; });
                __syncwarp();
                ct_fft_range<M, true, false, 32, SyncWarp, PosPad, 1, L, false>(B, lane, true, Z.tw, none, nonlin);
            }
        } else {
            ct_fft_range<M, true, false, 32, SyncWarp, PosPad, 0, L, false>(B, lane, true, Z.tw, none, nonlin);
        }
        __syncwarp();
    }

    if constexpr (SWEEP) {
        const int s = 1 + lane * LC;
        const int cnt = min(LC, NZ - 1 - s);              // unknowns of this lane's chunk (<= 0: idle lane)
        const int Gn = T.G;
        // table base of this lane: away from the left wall the elimination factors have converged to
        // their fixed point, so the interior chunks share one set of entries (T.gU, decided on the host
        // by a bitwise comparison) -- one broadcast address per load instead of 32 scattered ones
        const int sT = (lane >= T.gU && lane < Gn - 1) ? 1 + T.gU * LC : s;
        const bool l0 = lane == 0;
        auto t_inv = [&](int i) { if constexpr (CONSTTAB) return l0 ? P.inv0[i] : P.invU[i]; else return __ldg(&T.inv[sT + i]); };
        auto t_cc = [&](int i) { if constexpr (CONSTTAB) return l0 ? P.cc0[i] : P.ccU[i]; else return __ldg(&T.cc[sT + i]); };
        auto t_F = [&](int i) { if constexpr (CONSTTAB) return P.fU[i]; else return __ldg(&T.F[sT + i]); };
        auto t_Gm = [&](int i) { if constexpr (CONSTTAB) return l0 ? P.gm0[i] : P.gmU[i]; else return __ldg(&T.Gm[sT + i]); };
        // ---- A: local forward elimination with zero inflow; end nodes read as zero (R#7, R#8) ----
        cplx ev[LC];
        cplx e = mk(0.0, 0.0);
        {
            cplx pm = (lane == 0 || cnt <= 0) ? mk(0.0, 0.0) : A[PL::at(s - 1)];
            cplx p0 = (cnt > 0) ? A[PL::at(s)] : mk(0.0, 0.0);
#pragma unroll
            for (int i = 0; i < LC; ++i) {
                ev[i] = mk(0.0, 0.0);
                if (i < cnt) {
                    const int jn = s + i + 1;
                    const cplx pp = (jn < NZ - 1) ? A[PL::at(jn)] : mk(0.0, 0.0);
                    // inv_j (d_j + r e_{j-1}) = inv_j d_j + (-c_j) e_{j-1}: one dependent fma per unknown
                    cplx d = coef_mul(T.r, cadd(pm, pp));
                    d = coef_fma(T.omr2, p0, d);
                    e = coef_fma(coef_neg(t_cc(i)), e, coef_mul(t_inv(i), d));
                    ev[i] = e;
                    pm = p0;
                    p0 = pp;
                }
            }
        }
        // ---- B: forward inflow by a look-back over the lanes to the left ----
        const CT Ag = (lane < Gn) ? __ldg(&T.Ach[lane]) : ct_zero(CT());
        const CT Bg = (lane < Gn) ? __ldg(&T.Bch[lane]) : ct_zero(CT());
        cplx ein = mk(0.0, 0.0);
        for (int d = T.Kf; d >= 1; --d) {
            const int h = lane - d;
            const cplx Eh = shfl_c(e, h & 31);
            const CT Ah = shfl_ct(Ag, h & 31);
            if (h >= 0) ein = coef_fma(Ah, ein, Eh);
        }
        // ---- C: local back substitution with zero inflow ----
        cplx x = mk(0.0, 0.0);
#pragma unroll
        for (int i = LC - 1; i >= 0; --i) {
            if (i < cnt) {
                const cplx ee = coef_fma(t_F(i), ein, ev[i]);
                x = coef_fma(coef_neg(t_cc(i)), x, ee);
                ev[i] = x;
            }
        }
        // ---- D: backward inflow from the lanes to the right ----
        cplx xin = mk(0.0, 0.0);
        for (int d = T.Kb; d >= 1; --d) {
            const int h = lane + d;
            const cplx Xh = shfl_c(x, h & 31);
            const CT Bh = shfl_ct(Bg, h & 31);
            if (h < Gn) xin = coef_fma(Bh, xin, Xh);
        }
        __syncwarp();                                    // every lane has read its neighbours' values
        // ---- E: final values back into the line buffer; Dirichlet end nodes are exact zeros ----
#pragma unroll
        for (int i = 0; i < LC; ++i)
            if (i < cnt) A[PL::at(s + i)] = coef_fma(t_Gm(i), xin, ev[i]);
        if (lane == 0) A[PL::at(0)] = mk(0.0, 0.0);
        if (lane == 31) A[PL::at(NZ - 1)] = mk(0.0, 0.0);
        __syncwarp();
    }

    if constexpr (USE_A) {
#pragma unroll
        for (int i = 0; i < G::NPER; ++i) {
            const int e = 32 * i + lane;
            st_stream(p + e, A[PL::at(e)]);
        }
    }
}

}  // namespace dgpe
