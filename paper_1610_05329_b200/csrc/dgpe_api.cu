// dgpe_api.cu -- host side of libdgpe: the C-ABI of include/dgpe.h, the handle (plans, per-axis
// tables, workspace) and the kernel launches of one SSCN step.  No CPU implementation of any stage
// lives here: without a CUDA device every call fails.
#include "../../include/dgpe.h"

#include <algorithm>
#include <cmath>
#include <complex>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <map>
#include <mutex>
#include <tuple>
#include <utility>
#include <vector>

#include <cudaTypedefs.h>

#include "common.cuh"
#include "fft.cuh"
#include "observe.cuh"
#include "spectral.cuh"
#include "sweep.cuh"
#include "xyfft.cuh"
#include "xysweep.cuh"
#include "xysweep_tma.cuh"
#include "xyfft_tma.cuh"
#include "xyfft_pair.cuh"
#include "zline.cuh"

using namespace dgpe;

// ------------------------------------------------------------------------------------------------
// errors
// ------------------------------------------------------------------------------------------------
static thread_local char g_err[512] = "";

static int fail(int code, const char* fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
    return code;
}

#define CU(call)                                                                                   \
    do {                                                                                           \
        cudaError_t e_ = (call);                                                                   \
        if (e_ != cudaSuccess)                                                                     \
            return fail(e_ == cudaErrorMemoryAllocation ? DGPE_ERR_NOMEM : DGPE_ERR_CUDA,          \
                        "%s failed: %s", #call, cudaGetErrorString(e_));                           \
    } while (0)

extern "C" const char* dgpe_last_error(void) { return g_err; }

// ------------------------------------------------------------------------------------------------
// handle
// ------------------------------------------------------------------------------------------------
struct AxisSweep {
    int n = 0, Lc = 0, G = 0, Kf = 0, Kb = 0, gU = 0;
    std::complex<double> r;
    void* inv = nullptr;   // device tables, double (imag) or cplx (real)
    void* cc = nullptr;
    void* F = nullptr;
    void* Gm = nullptr;
    void* Ach = nullptr;
    void* Bch = nullptr;
    std::vector<std::complex<double>> h_inv, h_cc, h_F, h_Gm;   // host copies (kernel-parameter tables of the z sweep)
    bool consttab = false;   // chunk 0 + one converged chunk describe the whole line (zline.cuh ZTabs)
    void* ztab = nullptr;    // device, 8 Lc entries: [inv, cc, F, Gm] of chunk 0, then of the converged chunk (consttab only)
};

// defaults of k_fft_pair when the option is -1 (measured at 512^3: K3 0.677 -> 0.531 ms; K2/K4
// 0.408 -> 0.415 ms, so the y passes stay on k_fft_tma)
#ifndef DGPE_PAIR_DEFAULT_X
#define DGPE_PAIR_DEFAULT_X true
#define DGPE_PAIR_DEFAULT_Y false
#endif


enum { PF_Z = 1, PF_SWEEP_Y = 2, PF_SWEEP_X = 4, PF_FFT_Y = 8, PF_FFT_X = 16 };

struct dgpe_handle {
    int nx, ny, nz, nzh, mode;
    // DGPE_IMAG_RPSI (SV section 8f NEXT-2): mode is DGPE_IMAG, psi is nx*ny*nz plain doubles.  The x and y
    // sweeps act on the real and the imaginary part alike (real coefficients), so they run unchanged on psi
    // viewed as complex [nx][ny][nz/2]; nzc is that column count (nz in the complex modes).
    bool rpsi = false;
    int nzc = 0;
    double dx, dy, dz, dt, gamma, nu, lambda, g, gdd;
    long long N;
    // Slab views (dgpe_slab, SV section 8f NEXT-3; "data distributed along NX"): nx, ny above are the LOCAL extents
    // of the arrays this handle's kernels walk; the tables are those of the global grid gnx x gny x nz, entered at the
    // offsets x0, y0 of the slab.  A view holds whole lines along y (has_y: an x slab) or along x (has_x: a y slab).
    // Ordinary handles: gnx = nx, gny = ny, no offsets, both.
    int gnx = 0, gny = 0, x0 = 0, y0 = 0;
    bool has_x = true, has_y = true;
    bool own_spec = true;            // false: the half-spectrum buffer is handed in per call (y-slab view)
    double inv_ntot = 0.0;           // 1/(gnx gny nz): normalisation of the inverse transform (R#10)
    cudaStream_t stream = nullptr;
    int num_sms = 148;
    bool force_generic = false;      // DGPE_GENERIC=1: runtime-plan kernels only (A/B checks)
    int pf_mult = 1;                 // DGPE_PF_MULT: prefetch distance in units of one residency
    // L2 prefetch of the next residency, per kernel family (DGPE_PREFETCH=<mask> overrides, for A/B runs):
    // it pays for the z-line kernels and the y axis; on the x axis (row stride ny*nz) it costs time
    int prefetch = PF_Z | PF_SWEEP_Y | PF_FFT_Y;
    bool use_tma_fft = true;         // DGPE_TMA_FFT=0: K2/K4 load and store through the threads (k_fft_xy)
    // K3 on the TMA pipeline (k_fft_tma_xudd): measured 1.98 -> 1.45 ms at nx = 768 (one 768-thread CTA per SM
    // otherwise), 0.67 -> 0.70 ms at nx = 512, so by default from nx = 640 up; DGPE_TMA_K3=0|1: never | every length
    int use_tma_k3 = -1;
    bool use_tma_x = false;          // DGPE_TMA=2: TMA on the x axis at every length (A/B)
    bool use_tma = true;             // DGPE_TMA=0: the x/y sweeps load and store through the threads (k_sweep_xy)
    bool zfast = false;              // warp-per-line z kernels (zline.cuh) and the fused step order z, x, y
    dgpe_options opt;                // as given to dgpe_create_ex (all -1 from dgpe_create)
    int device = 0;                  // the CUDA device the handle lives on (current at creation)

    cplx* spec = nullptr;                       // [nx][ny][nzh]
    FftPlan plan_x{}, plan_y{}, plan_zh{};      // transform lengths nx, ny, nz/2
    cplx *tw_x = nullptr, *tw_y = nullptr, *tw_zh = nullptr, *tw_split = nullptr;
    double *kx2 = nullptr, *ky2 = nullptr, *kz2 = nullptr;
    double *vx = nullptr, *vy = nullptr, *vz = nullptr;      // gamma^2 x^2, nu^2 y^2, lambda^2 z^2
    double *x2 = nullptr, *y2 = nullptr, *z2 = nullptr;      // squared coordinates
    AxisSweep sw[3];
    double* scal = nullptr;          // device scalars (SC_*)
    double* partials = nullptr;
    unsigned int* ticket = nullptr;
    double* d_out = nullptr;         // device results (16 doubles)
    double* h_out = nullptr;         // pinned host mirror
    cplx* psi_stage = nullptr;       // dgpe_step_host: device copy of psi (lazy)
    // CUDA graph of one step (7 or 8 kernel nodes), captured once per psi pointer on a private stream and
    // replayed on the handle's stream: removes the per-launch host cost that dominates the small grids
    bool use_graph = true;           // DGPE_GRAPH=0: plain launches
    bool warmed = false;             // one eager step has run (lazy per-kernel attribute setup done)
    cudaStream_t cap_stream = nullptr;
    // one instantiated graph per psi pointer, most recently used first (ping-pong buffers, dgpe_step after
    // dgpe_step_host, ... keep their graphs)
    std::vector<std::pair<cplx*, cudaGraphExec_t>> step_execs;
    std::vector<cudaEvent_t> prof_ev; // dgpe_step_profile
    std::vector<void*> owned;        // everything to cudaFree
};

static bool z_specialised(int nz);

static int threads_for(int nbf)
{
    int t = nbf * TILE_COLS;
    return ((t + 31) / 32) * 32;
}

template <typename T>
static int upload(dgpe_handle* h, const std::vector<T>& v, T** out)
{
    T* d = nullptr;
    CU(cudaMalloc(&d, sizeof(T) * (v.empty() ? 1 : v.size())));
    h->owned.push_back(d);
    if (!v.empty()) CU(cudaMemcpy(d, v.data(), sizeof(T) * v.size(), cudaMemcpyHostToDevice));
    *out = d;
    return DGPE_OK;
}

// FFT-friendly sizes: 2^a 3^b 5^c 7^d 11^e 13^f
static bool smooth2357(int n)
{
    if (n < 1) return false;
    for (int f : {2, 3, 5, 7, 11, 13})
        while (n % f == 0) n /= f;
    return n == 1;
}

// radices 8, 4, 2 first, then 3, 5, 7, 11, 13; butterfly slots per column = n / largest radix
static int make_plan(dgpe_handle* h, int n, FftPlan* P, cplx** tw_dev, int max_slots)
{
    std::memset(P, 0, sizeof(*P));
    P->n = n;
    int m = n, np = 0, rmax = 1;
    const int order[8] = {8, 4, 2, 3, 5, 7, 11, 13};
    for (int oi = 0; oi < 8; ++oi) {
        const int R = order[oi];
        while (m % R == 0 && m > 1) {
            if (np >= MAX_PASSES) return fail(DGPE_ERR_UNSUPPORTED, "FFT length %d needs too many passes", n);
            P->radix[np++] = R;
            m /= R;
            if (R > rmax) rmax = R;
        }
    }
    if (m != 1) return fail(DGPE_ERR_ARG, "FFT length %d is not of the form 2^a 3^b 5^c 7^d 11^e 13^f", n);
    if (np == 0) {           // n == 1: one radix-1 "pass" does not exist; callers never ask for it
        return fail(DGPE_ERR_ARG, "FFT length %d too small", n);
    }
    P->npass = np;
    // butterfly slots per line: n / (largest radix, at most 8) -- a slot then runs at most ceil(8/R) butterflies
    // of a radix-R pass (radices 11 and 13 leave some slots idle) -- bounded by the kernel's thread limit
    const int rdiv = std::min(rmax, 8);
    P->nbf = std::min((n + rdiv - 1) / rdiv, max_slots);
    for (int p = 0; p < np; ++p) {
        const int nbut = n / P->radix[p];
        P->nb[p] = (nbut + P->nbf - 1) / P->nbf;
    }
    std::vector<cplx> tw(n);
    const long double TWO_PI = 6.283185307179586476925286766559005768L;
    for (int j = 0; j < n; ++j) {
        long double a = TWO_PI * (long double)j / (long double)n;
        tw[j] = make_double2((double)cosl(a), (double)(-sinl(a)));
    }
    int rc = upload(h, tw, tw_dev);
    P->tw = *tw_dev;
    return rc;
}

// wave number of DFT bin m (R#10, R#11): k = 2 pi f/(n d), f = m for m <= n/2, else m - n
static std::vector<double> wavenum_sq(int n, double d, int count)
{
    const double PI = 3.14159265358979323846264338327950288;
    std::vector<double> v(count);
    for (int m = 0; m < count; ++m) {
        int f = (m <= n / 2) ? m : m - n;
        double k = 2.0 * PI * (double)f / ((double)n * d);
        v[m] = k * k;
    }
    return v;
}

template <typename CT>
static CT to_ct(std::complex<double> z);
template <>
double to_ct<double>(std::complex<double> z) { return z.real(); }
template <>
cplx to_ct<cplx>(std::complex<double> z) { return make_double2(z.real(), z.imag()); }

template <typename CT>
static int build_sweep(dgpe_handle* h, AxisSweep* S, int n, std::complex<double> r, int lc)
{
    typedef std::complex<double> C;
    S->n = n;
    S->r = r;
    S->Lc = lc;
    const int nun = n - 2;
    S->G = (nun + S->Lc - 1) / S->Lc;
    std::vector<C> inv(n, C(0)), cc(n, C(0)), F(n, C(0)), Gm(n, C(0)), A(S->G, C(0)), B(S->G, C(0));
    const C diag = 1.0 + 2.0 * r;
    inv[1] = 1.0 / diag;
    cc[1] = -r * inv[1];
    for (int j = 2; j <= n - 2; ++j) {
        inv[j] = 1.0 / (diag + r * cc[j - 1]);
        cc[j] = -r * inv[j];
    }
    double amax = 0.0, bmax = 0.0;
    for (int g = 0; g < S->G; ++g) {
        const int s = 1 + g * S->Lc, t = std::min(s + S->Lc, n - 1);
        C acc = 1.0;
        for (int j = s; j < t; ++j) { acc *= r * inv[j]; F[j] = acc; }
        A[g] = acc;
        acc = 1.0;
        for (int j = t - 1; j >= s; --j) { acc *= -cc[j]; Gm[j] = acc; }
        B[g] = acc;
        amax = std::max(amax, std::abs(A[g]));
        bmax = std::max(bmax, std::abs(B[g]));
    }
    // first chunk from which all full interior chunks (.. G-2) carry bit-identical table entries
    S->gU = S->G;
    for (int c0 = 0; c0 + 1 < S->G; ++c0) {
        bool same = true;
        for (int g = c0 + 1; g <= S->G - 2 && same; ++g)
            for (int i = 0; i < S->Lc && same; ++i) {
                const int a = 1 + c0 * S->Lc + i, b = 1 + g * S->Lc + i;
                same = inv[a] == inv[b] && cc[a] == cc[b] && F[a] == F[b] && Gm[a] == Gm[b];
            }
        if (same) { S->gU = c0; break; }
    }
    S->consttab = (S->G == 1);
    if (S->G >= 2 && S->gU <= 1) {
        bool same = true;
        const int g = S->G - 1;
        for (int i = 0; i < S->Lc && 1 + g * S->Lc + i <= n - 2 && same; ++i) {
            const int a = 1 + S->Lc + i, b = 1 + g * S->Lc + i;
            same = inv[a] == inv[b] && cc[a] == cc[b] && F[a] == F[b];
        }
        S->consttab = same;
    }
    S->h_inv = inv; S->h_cc = cc; S->h_F = F; S->h_Gm = Gm;
    const double tol = std::ldexp(1.0, -80);
    auto depth = [&](double q) {
        int K = 1;
        double p = q;
        while (K < S->G && p > tol) { p *= q; ++K; }
        return K;
    };
    S->Kf = depth(amax);
    S->Kb = depth(bmax);
    auto conv = [&](const std::vector<C>& v, void** out) -> int {
        std::vector<CT> w(v.size());
        for (size_t i = 0; i < v.size(); ++i) w[i] = to_ct<CT>(v[i]);
        CT* d = nullptr;
        int rc = upload(h, w, &d);
        *out = d;
        return rc;
    };
    int rc;
    if ((rc = conv(inv, &S->inv))) return rc;
    if ((rc = conv(cc, &S->cc))) return rc;
    if ((rc = conv(F, &S->F))) return rc;
    if ((rc = conv(Gm, &S->Gm))) return rc;
    if ((rc = conv(A, &S->Ach))) return rc;
    if ((rc = conv(B, &S->Bch))) return rc;
    if (S->consttab) {
        const int lc2 = S->Lc, u0 = (S->G >= 2) ? 1 + lc2 : 1;
        std::vector<C> zt(8 * (size_t)lc2, C(0));
        for (int i = 0; i < lc2; ++i) {
            const int a = std::min(1 + i, n - 1), b = std::min(u0 + i, n - 1);      // entries past n-2 are zero and unused
            zt[i] = inv[a]; zt[lc2 + i] = cc[a]; zt[2 * lc2 + i] = F[b]; zt[3 * lc2 + i] = Gm[a];
            zt[4 * lc2 + i] = inv[b]; zt[5 * lc2 + i] = cc[b]; zt[6 * lc2 + i] = F[b]; zt[7 * lc2 + i] = Gm[b];
        }
        if ((rc = conv(zt, &S->ztab))) return rc;
    }
    return DGPE_OK;
}

static size_t sweep_smem(int n, int G, bool zaxis)
{
    return sizeof(cplx) * ((size_t)n * (zaxis ? 9 : 8) + 2 * (size_t)G * TILE_COLS);
}

// Per (kernel, device) setup that must precede a launch with more than 48 KB of dynamic shared memory,
// and the resident CTAs per SM of that launch shape.  Cached: the kernels are launched thousands of
// times; keyed by device so that one process may hold handles on several GPUs; guarded for threads.
static int kernel_setup(const void* func, int threads, size_t smem, int* ctas_per_sm)
{
    static std::mutex mu;
    static std::map<std::pair<const void*, int>, size_t> allowed;                              // (kernel, device) -> opt-in bytes
    static std::map<std::tuple<const void*, int, int, size_t>, int> resident;                  // + (threads, bytes) -> CTAs per SM
    if (smem > 227 * 1024) return fail(DGPE_ERR_UNSUPPORTED, "a kernel needs %zu bytes of shared memory", smem);
    int dev = 0;
    CU(cudaGetDevice(&dev));
    std::lock_guard<std::mutex> lock(mu);
    size_t& optin = allowed[std::make_pair(func, dev)];
    // (the limit counts static shared memory too: opt in from 40 KB of dynamic memory up)
    if (smem > 40 * 1024 && smem > optin) {
        CU(cudaFuncSetAttribute(func, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        optin = smem;
    }
    int& n = resident[std::make_tuple(func, dev, threads, smem)];
    if (!n) {
        CU(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, func, threads, smem));
        if (n < 1) return fail(DGPE_ERR_CUDA, "a kernel does not fit on an SM (%d threads, %zu bytes of shared memory)", threads, smem);
    }
    if (ctas_per_sm) *ctas_per_sm = n;
    return DGPE_OK;
}

static int init_handle(dgpe_handle* h)
{
    const int nx = h->nx, ny = h->ny, nz = h->nz, nzh = h->nzh, M = nz / 2;
    int rc;
    int dev_count = 0;
    CU(cudaGetDeviceCount(&dev_count));
    if (dev_count < 1) return fail(DGPE_ERR_CUDA, "no CUDA device");
    {
        int dev = 0;
        CU(cudaGetDevice(&dev));
        h->device = dev;
        CU(cudaDeviceGetAttribute(&h->num_sms, cudaDevAttrMultiProcessorCount, dev));
        // options (dgpe_create_ex; -1 = default): A/B switches and in-repo cross-checks, never read from the environment
        const dgpe_options& o = h->opt;
        h->force_generic = o.generic == 1;
        h->zfast = !h->force_generic && z_specialised(nz);
        if (h->rpsi && !h->zfast)
            return fail(DGPE_ERR_UNSUPPORTED, "DGPE_IMAG_RPSI needs one of the specialised z lengths (nz = %d is not)", nz);
        if (o.prefetch >= 0) h->prefetch = o.prefetch;
        h->use_tma = o.tma != 0;
        h->use_tma_x = o.tma == 2;
        h->use_tma_fft = h->use_tma && o.tma_fft != 0;
        h->use_tma_k3 = !h->use_tma ? 0 : (o.tma_k3 == 1) ? 1 : (o.tma_k3 == 0) ? 0 : -1;
        h->use_graph = o.graph != 0;
        if (o.pf_mult > 0) h->pf_mult = o.pf_mult;
    }

    if (!h->gnx) { h->gnx = nx; h->gny = ny; }
    const int gnx = h->gnx, gny = h->gny;
    h->inv_ntot = 1.0 / ((double)gnx * (double)gny * (double)nz);
    if (h->has_x && (rc = make_plan(h, nx, &h->plan_x, &h->tw_x, 128))) return rc;
    if (h->has_y && (rc = make_plan(h, ny, &h->plan_y, &h->tw_y, 128))) return rc;
    if ((rc = make_plan(h, M, &h->plan_zh, &h->tw_zh, 64))) return rc;
    {
        std::vector<cplx> tw(M + 1);
        const long double TWO_PI = 6.283185307179586476925286766559005768L;
        for (int k = 0; k <= M; ++k) {
            long double a = TWO_PI * (long double)k / (long double)nz;
            tw[k] = make_double2((double)cosl(a), (double)(-sinl(a)));
        }
        if ((rc = upload(h, tw, &h->tw_split))) return rc;
    }
    if ((rc = upload(h, wavenum_sq(gnx, h->dx, gnx), &h->kx2))) return rc;
    if ((rc = upload(h, wavenum_sq(gny, h->dy, gny), &h->ky2))) return rc;
    if ((rc = upload(h, wavenum_sq(nz, h->dz, nzh), &h->kz2))) return rc;
    h->kx2 += h->x0;      // tables of the global grid, entered at the slab's offset (the uploads stay owned at their bases)
    h->ky2 += h->y0;

    auto coord_tables = [&](int n, double d, double om, double** v, double** c2) -> int {
        std::vector<double> tv(n), tc(n);
        for (int i = 0; i < n; ++i) {
            double x = (double)(i - n / 2) * d;      // R#6
            tv[i] = om * om * x * x;
            tc[i] = x * x;
        }
        int r1 = upload(h, tv, v);
        if (r1) return r1;
        return upload(h, tc, c2);
    };
    if ((rc = coord_tables(gnx, h->dx, h->gamma, &h->vx, &h->x2))) return rc;
    if ((rc = coord_tables(gny, h->dy, h->nu, &h->vy, &h->y2))) return rc;
    if ((rc = coord_tables(nz, h->dz, h->lambda, &h->vz, &h->z2))) return rc;
    h->vx += h->x0; h->x2 += h->x0;
    h->vy += h->y0; h->y2 += h->y0;

    const int ns[3] = {nx, ny, nz};
    const double ds[3] = {h->dx, h->dy, h->dz};
    for (int a = 0; a < 3; ++a) {
        if ((a == 0 && !h->has_x) || (a == 1 && !h->has_y)) continue;      // a slab view never sweeps along its cut axis
        const double rr = h->dt / (4.0 * ds[a] * ds[a]);      // R#9
        // chunk length of the sweep recursions: 8 (or 16) unknowns per thread on the strided axes; on z
        // the warp-per-line kernel gives every lane ceil((nz-2)/32) unknowns
        int lc = (ns[a] <= 770 && !h->force_generic) ? 8 : 16;
        if (a == 2 && !h->zfast) lc = 16;      // generic z kernel: 8 * G <= 512 threads
        if (a == 2 && h->zfast) lc = ((nz - 2 + z_team(nz) - 1) / z_team(nz)) | 1;      // = ZGeom<nz>::LC, odd (zline.cuh)
        if (h->mode == DGPE_IMAG)
            rc = build_sweep<double>(h, &h->sw[a], ns[a], std::complex<double>(rr, 0.0), lc);
        else
            rc = build_sweep<cplx>(h, &h->sw[a], ns[a], std::complex<double>(0.0, rr), lc);
        if (rc) return rc;
    }

    if (h->own_spec) {
        CU(cudaMalloc(&h->spec, sizeof(cplx) * (size_t)nx * ny * nzh));
        h->owned.push_back(h->spec);
    }
    size_t nblk = std::max({(size_t)(((long long)ny * nz + 7) / 8), (size_t)nx * ((nz + 7) / 8),
                            (size_t)(((long long)nx * ny + 7) / 8), (size_t)4096});
    CU(cudaMalloc(&h->partials, sizeof(double) * nblk * MAX_RED));
    h->owned.push_back(h->partials);
    CU(cudaMalloc(&h->ticket, sizeof(unsigned int)));
    h->owned.push_back(h->ticket);
    CU(cudaMemset(h->ticket, 0, sizeof(unsigned int)));
    CU(cudaMalloc(&h->scal, sizeof(double) * SC_COUNT));
    h->owned.push_back(h->scal);
    {
        double init[SC_COUNT] = {1.0, 1.0, 1.0, 0.0, 0, 0, 0, 0};
        CU(cudaMemcpy(h->scal, init, sizeof(init), cudaMemcpyHostToDevice));
    }
    CU(cudaMalloc(&h->d_out, sizeof(double) * 16));
    h->owned.push_back(h->d_out);
    CU(cudaMallocHost(&h->h_out, sizeof(double) * 16));

    return DGPE_OK;
}

static thread_local int g_err_code = DGPE_OK;

extern "C" int dgpe_last_error_code(void) { return g_err_code; }

extern "C" dgpe_handle* dgpe_create_ex(int nx, int ny, int nz, double dx, double dy, double dz, double dt,
                                       double gamma, double nu, double lambda, double g, double gdd, int mode,
                                       const dgpe_options* opt)
{
    g_err[0] = 0;
    g_err_code = DGPE_OK;
    auto bad = [](int code) -> dgpe_handle* { g_err_code = code; return nullptr; };
    const int ns[3] = {nx, ny, nz};
    for (int a = 0; a < 3; ++a) {
        if (ns[a] < 4) return bad(fail(DGPE_ERR_ARG, "grid size %d < 4", ns[a]));
        if (!smooth2357(ns[a])) return bad(fail(DGPE_ERR_ARG, "grid size %d is not of the form 2^a 3^b 5^c 7^d 11^e 13^f", ns[a]));
        if (ns[a] > DGPE_MAX_N) return bad(fail(DGPE_ERR_UNSUPPORTED, "grid size %d > %d", ns[a], DGPE_MAX_N));
    }
    if (nz % 2) return bad(fail(DGPE_ERR_ARG, "nz = %d must be even", nz));
    if (!(dx > 0.0) || !(dy > 0.0) || !(dz > 0.0) || !(dt > 0.0) || !std::isfinite(dx) || !std::isfinite(dy) ||
        !std::isfinite(dz) || !std::isfinite(dt))
        return bad(fail(DGPE_ERR_ARG, "dx, dy, dz, dt must be positive and finite"));
    if (mode != DGPE_IMAG && mode != DGPE_REAL && mode != DGPE_IMAG_RPSI)
        return bad(fail(DGPE_ERR_ARG, "mode %d is none of DGPE_IMAG, DGPE_REAL, DGPE_IMAG_RPSI", mode));
    dgpe_handle* h = new (std::nothrow) dgpe_handle();
    if (!h) return bad(fail(DGPE_ERR_NOMEM, "host allocation failed"));
    if (opt) h->opt = *opt;
    else { int* f = reinterpret_cast<int*>(&h->opt); for (size_t i = 0; i < sizeof(dgpe_options) / sizeof(int); ++i) f[i] = -1; }
    h->nx = nx; h->ny = ny; h->nz = nz; h->nzh = nz / 2 + 1;
    h->rpsi = mode == DGPE_IMAG_RPSI;
    h->mode = h->rpsi ? DGPE_IMAG : mode;
    h->nzc = h->rpsi ? nz / 2 : nz;
    h->dx = dx; h->dy = dy; h->dz = dz; h->dt = dt;
    h->gamma = gamma; h->nu = nu; h->lambda = lambda; h->g = g; h->gdd = gdd;
    h->N = (long long)nx * ny * nz;
    const int rc = init_handle(h);
    if (rc != DGPE_OK) {
        char keep[sizeof(g_err)];
        std::memcpy(keep, g_err, sizeof(keep));
        dgpe_destroy(h);
        std::memcpy(g_err, keep, sizeof(keep));
        return bad(rc);
    }
    return h;
}

extern "C" dgpe_handle* dgpe_create(int nx, int ny, int nz, double dx, double dy, double dz, double dt,
                                    double gamma, double nu, double lambda, double g, double gdd, int mode)
{
    return dgpe_create_ex(nx, ny, nz, dx, dy, dz, dt, gamma, nu, lambda, g, gdd, mode, nullptr);
}

extern "C" void dgpe_destroy(dgpe_handle* h)
{
    if (!h) return;
    cudaStreamSynchronize(h->stream);
    for (auto& e : h->step_execs) cudaGraphExecDestroy(e.second);
    if (h->cap_stream) cudaStreamDestroy(h->cap_stream);
    for (void* p : h->owned) cudaFree(p);
    if (h->h_out) cudaFreeHost(h->h_out);
    for (cudaEvent_t e : h->prof_ev) cudaEventDestroy(e);
    delete h;
}

extern "C" int dgpe_set_stream(dgpe_handle* h, void* cuda_stream)
{
    if (!h) return fail(DGPE_ERR_ARG, "NULL handle");
    h->stream = (cudaStream_t)cuda_stream;
    return DGPE_OK;
}

extern "C" int dgpe_synchronize(dgpe_handle* h)
{
    if (!h) return fail(DGPE_ERR_ARG, "NULL handle");
    CU(cudaStreamSynchronize(h->stream));
    return DGPE_OK;
}

// ------------------------------------------------------------------------------------------------
// launches
// ------------------------------------------------------------------------------------------------
// every call must run with the handle's device current (kernels, tensor maps and pointers belong to it)
static int check_device(const dgpe_handle* h)
{
    int dev = -1;
    CU(cudaGetDevice(&dev));
    if (dev != h->device)
        return fail(DGPE_ERR_ARG, "the handle lives on CUDA device %d but device %d is current", h->device, dev);
    return DGPE_OK;
}

static int check_launch(const char* what)
{
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(DGPE_ERR_CUDA, "launch of %s failed: %s", what, cudaGetErrorString(e));
    return DGPE_OK;
}

// ------------------------------------------------------------------------------------------------
// warp-per-line z kernels (zline.cuh): specialised line lengths
// ------------------------------------------------------------------------------------------------
#define DGPE_Z_SIZES(X) X(64) X(128) X(160) X(192) X(240) X(250) X(256) X(320) X(384) X(480) X(500) X(512) X(640) X(768)

static bool z_specialised(int nz)
{
    switch (nz) {
#define X(NN) case NN:
        DGPE_Z_SIZES(X)
#undef X
        return true;
        default: return false;
    }
}

// kernel-parameter copy of the sweep tables: chunk 0 and the converged chunk (sweep.cuh ChunkTabs)
template <typename CT, int LC>
static void fill_chunk_tabs(const AxisSweep& S, bool use, ChunkTabs<CT, LC>* P)
{
    std::memset(P, 0, sizeof(*P));
    if (!use) return;
    const int n = S.n, u0 = (S.G >= 2) ? 1 + LC : 1;
    for (int i = 0; i < LC; ++i) {
        const int a = std::min(1 + i, n - 1), b = std::min(u0 + i, n - 1);     // entries past n-2 are zero and unused
        P->inv0[i] = to_ct<CT>(S.h_inv[a]); P->cc0[i] = to_ct<CT>(S.h_cc[a]); P->gm0[i] = to_ct<CT>(S.h_Gm[a]);
        P->invU[i] = to_ct<CT>(S.h_inv[b]); P->ccU[i] = to_ct<CT>(S.h_cc[b]);
        P->fU[i] = to_ct<CT>(S.h_F[b]); P->gmU[i] = to_ct<CT>(S.h_Gm[b]);
    }
}

#ifndef DGPE_ZCAP_RPSI
#define DGPE_ZCAP_RPSI 20      // measured at 512^3: 16 -> 0.758 ms, 20 -> 0.733 ms, 24 -> 0.773 ms
#endif
constexpr int Z_MAIN_WARPS = 1;      // warps per CTA of k_z_main: one, so that a finished line frees its slot at once

template <int NZ>
constexpr int z_main_minb(bool use_a, bool use_b, int a_size)
{
    const int per_cta = Z_MAIN_WARPS * ZGeom<NZ>::LPW * ((use_a ? ZGeom<NZ>::A_ELEMS * a_size : 0) + (use_b ? ZGeom<NZ>::B_ELEMS * 16 : 0)) + 1024;
    // 16 warps per SM: 128 registers per thread; the real-valued sweep needs half the registers of the complex one
    const int m = (227 * 1024) / per_cta, cap = (a_size == 8 ? DGPE_ZCAP_RPSI : 16) / Z_MAIN_WARPS;
    return m < 1 ? 1 : (m > cap ? cap : m);
}

template <int NZ>
static int launch_z_r2c_n(dgpe_handle* h, const cplx* psi)
{
    constexpr int WARPS = 1;                             // one warp per CTA: a finished line frees its slot at once
    constexpr int LINES = WARPS * ZGeom<NZ>::LPW;        // lines per CTA
    const size_t smem = (size_t)LINES * ZGeom<NZ>::B_ELEMS * sizeof(cplx);
    const int nlines = h->nx * h->ny;
    if (h->rpsi) {
        auto kern = k_z_r2c<NZ, WARPS, double>;
        int rc = kernel_setup((const void*)kern, 32 * WARPS, smem, nullptr);
        if (rc) return rc;
        kern<<<(nlines + LINES - 1) / LINES, 32 * WARPS, smem, h->stream>>>((const double*)psi, h->spec, nlines, h->tw_zh,
                                                                            h->tw_split, h->scal);
        return check_launch("k_z_r2c");
    }
    auto kern = k_z_r2c<NZ, WARPS, cplx>;
    int rc = kernel_setup((const void*)kern, 32 * WARPS, smem, nullptr);
    if (rc) return rc;
    kern<<<(nlines + LINES - 1) / LINES, 32 * WARPS, smem, h->stream>>>(psi, h->spec, nlines, h->tw_zh, h->tw_split, h->scal);
    return check_launch("k_z_r2c");
}

template <int NZ, typename CT, typename DT, int SPEC, bool SWEEP, bool CONSTTAB>
static int launch_z_main_c(dgpe_handle* h, cplx* psi, double* phi_out)
{
    constexpr int WARPS = Z_MAIN_WARPS, LC = ZGeom<NZ>::LC, LINES = WARPS * ZGeom<NZ>::LPW;
    constexpr bool USE_A = SPEC != ZS_PHI, USE_B = SPEC != ZS_NONE;
    constexpr int MINB = z_main_minb<NZ>(USE_A, USE_B, (int)sizeof(DT));
    const size_t smem = (size_t)LINES * ((USE_A ? ZGeom<NZ>::A_ELEMS * sizeof(DT) : 0) + (USE_B ? ZGeom<NZ>::B_ELEMS * sizeof(cplx) : 0));
    auto kern = k_z_main<NZ, CT, DT, SPEC, SWEEP, CONSTTAB, WARPS, MINB>;
    int ctas_per_sm = 0;
    int rc = kernel_setup((const void*)kern, 32 * WARPS, smem, &ctas_per_sm);
    if (rc) return rc;
    const AxisSweep& S = h->sw[2];
    SweepTables<CT> T;
    T.r = to_ct<CT>(S.r);
    T.omr2 = to_ct<CT>(1.0 - 2.0 * S.r);
    T.inv = (const CT*)S.inv; T.cc = (const CT*)S.cc; T.F = (const CT*)S.F; T.Gm = (const CT*)S.Gm;
    T.Ach = (const CT*)S.Ach; T.Bch = (const CT*)S.Bch; T.ztab = (const CT*)S.ztab;
    T.Lc = S.Lc; T.G = S.G; T.Kf = S.Kf; T.Kb = S.Kb; T.gU = S.gU;
    if (SWEEP && (S.Lc != LC || S.G > ZGeom<NZ>::T)) return fail(DGPE_ERR_CUDA, "z sweep tables do not match the z-line kernel");
    ChunkTabs<CT, LC> P;
    fill_chunk_tabs<CT, LC>(S, SWEEP && CONSTTAB && sizeof(DT) == sizeof(double), &P);      // real-valued psi only (zline.cuh)
    ZMainArgs Z;
    Z.nlines = h->nx * h->ny; Z.ny = h->ny;
    Z.dt = h->dt; Z.g = h->g; Z.gdd = h->gdd;
    Z.vx = h->vx; Z.vy = h->vy;
    Z.dz = h->dz; Z.lam2 = h->lambda * h->lambda;
    Z.scal = h->scal; Z.tw = h->tw_zh; Z.tws = h->tw_split; Z.phi_out = phi_out;
    Z.pf_lines = (h->prefetch & PF_Z) ? h->pf_mult * ctas_per_sm * h->num_sms * LINES : 0;
    if (SWEEP && CONSTTAB && !S.ztab) return fail(DGPE_ERR_CUDA, "z sweep tables were not built for the z-line kernel");
    kern<<<(Z.nlines + LINES - 1) / LINES, 32 * WARPS, smem, h->stream>>>((DT*)psi, h->spec, Z, T, (const CT*)S.ztab, P);
    return check_launch("k_z_main");
}

template <int NZ, typename CT, typename DT, int SPEC, bool SWEEP>
static int launch_z_main_n(dgpe_handle* h, cplx* psi, double* phi_out)
{
    if constexpr (SWEEP) {
        if (h->sw[2].consttab) return launch_z_main_c<NZ, CT, DT, SPEC, true, true>(h, psi, phi_out);
    }
    return launch_z_main_c<NZ, CT, DT, SPEC, SWEEP, false>(h, psi, phi_out);
}

// what: 0 = C2R + nonlinear, 1 = C2R + nonlinear + z sweep, 2 = z sweep only, 3 = C2R -> phi_out
template <int NZ>
static int launch_z_main_nz(dgpe_handle* h, cplx* psi, int what, double* phi_out)
{
    const bool imag = h->mode == DGPE_IMAG;
    if (h->rpsi) {      // real-valued psi (psi points to doubles); ZS_PHI does not touch psi
        switch (what) {
            case 0: return launch_z_main_n<NZ, double, double, ZS_IMAG, false>(h, psi, nullptr);
            case 1: return launch_z_main_n<NZ, double, double, ZS_IMAG, true>(h, psi, nullptr);
            case 2: return launch_z_main_n<NZ, double, double, ZS_NONE, true>(h, psi, nullptr);
            default: break;
        }
    }
    switch (what) {
        case 0: return imag ? launch_z_main_n<NZ, double, cplx, ZS_IMAG, false>(h, psi, nullptr)
                            : launch_z_main_n<NZ, cplx, cplx, ZS_REAL, false>(h, psi, nullptr);
        case 1: return imag ? launch_z_main_n<NZ, double, cplx, ZS_IMAG, true>(h, psi, nullptr)
                            : launch_z_main_n<NZ, cplx, cplx, ZS_REAL, true>(h, psi, nullptr);
        case 2: return imag ? launch_z_main_n<NZ, double, cplx, ZS_NONE, true>(h, psi, nullptr)
                            : launch_z_main_n<NZ, cplx, cplx, ZS_NONE, true>(h, psi, nullptr);
        default: return launch_z_main_n<NZ, double, cplx, ZS_PHI, false>(h, psi, phi_out);
    }
}

static int launch_z_main(dgpe_handle* h, cplx* psi, int what, double* phi_out)
{
    switch (h->nz) {
#define X(NN) case NN: return launch_z_main_nz<NN>(h, psi, what, phi_out);
        DGPE_Z_SIZES(X)
#undef X
        default: return fail(DGPE_ERR_UNSUPPORTED, "no z-line kernel for nz = %d", h->nz);
    }
}

static int launch_z_r2c(dgpe_handle* h, const cplx* psi)
{
    switch (h->nz) {
#define X(NN) case NN: return launch_z_r2c_n<NN>(h, psi);
        DGPE_Z_SIZES(X)
#undef X
        default: return fail(DGPE_ERR_UNSUPPORTED, "no z-line kernel for nz = %d", h->nz);
    }
}

// ---- K1 ----
static int launch_k1(dgpe_handle* h, const cplx* psi)
{
    if (h->zfast) return launch_z_r2c(h, psi);
    const int nlines = h->nx * h->ny, M = h->nz / 2;
    const int thr = threads_for(h->plan_zh.nbf);
    const size_t sm = sizeof(cplx) * TILE_COLS * (size_t)M;
    int rcs = kernel_setup((const void*)k_dens_r2c, thr, sm, nullptr);
    if (rcs) return rcs;
    k_dens_r2c<<<(nlines + 7) / 8, thr, sm, h->stream>>>(psi, h->spec, nlines, h->nz, h->plan_zh, h->tw_split, h->scal);
    return check_launch("k_dens_r2c");
}

// ---- K2 / K4 (axis 1) and K3 (axis 0): pipelined compile-time kernels when the length is one of the
// specialised sizes, else the generic runtime-plan kernels ----
template <int N, int KIND>
static int launch_fft_xy_n(dgpe_handle* h, const LineMap& map, int nbatch, const cplx* tw)
{
    const size_t smem = (size_t)N * TILE_COLS * sizeof(cplx);
    auto kern = k_fft_xy<N, KIND>;
    int ctas_per_sm = 0;
    int rc = kernel_setup((const void*)kern, xy_threads<N>(), smem, &ctas_per_sm);
    if (rc) return rc;
    UddArgs U{h->nzh, h->kx2, h->ky2, h->kz2, 2.0 * 3.14159265358979323846264338327950288 / ((double)h->nx * h->dx), h->inv_ntot,
              (h->prefetch & (KIND == FFT_X_UDD ? PF_FFT_X : PF_FFT_Y)) ? h->pf_mult * ctas_per_sm * h->num_sms : 0};
    dim3 grid((map.ncols + TILE_COLS - 1) / TILE_COLS, nbatch);
    kern<<<grid, xy_threads<N>(), smem, h->stream>>>(h->spec, map, tw, U);
    return check_launch("k_fft_xy");
}

template <int KIND>
static int launch_fft_xy(dgpe_handle* h, int n, const LineMap& map, int nbatch, const cplx* tw, bool* handled)
{
    *handled = true;
    switch (n) {
        case 8: return launch_fft_xy_n<8, KIND>(h, map, nbatch, tw);
        case 16: return launch_fft_xy_n<16, KIND>(h, map, nbatch, tw);
        case 32: return launch_fft_xy_n<32, KIND>(h, map, nbatch, tw);
        case 48: return launch_fft_xy_n<48, KIND>(h, map, nbatch, tw);
        case 64: return launch_fft_xy_n<64, KIND>(h, map, nbatch, tw);
        case 96: return launch_fft_xy_n<96, KIND>(h, map, nbatch, tw);
        case 128: return launch_fft_xy_n<128, KIND>(h, map, nbatch, tw);
        case 160: return launch_fft_xy_n<160, KIND>(h, map, nbatch, tw);
        case 192: return launch_fft_xy_n<192, KIND>(h, map, nbatch, tw);
        case 240: return launch_fft_xy_n<240, KIND>(h, map, nbatch, tw);
        case 256: return launch_fft_xy_n<256, KIND>(h, map, nbatch, tw);
        case 320: return launch_fft_xy_n<320, KIND>(h, map, nbatch, tw);
        case 384: return launch_fft_xy_n<384, KIND>(h, map, nbatch, tw);
        case 480: return launch_fft_xy_n<480, KIND>(h, map, nbatch, tw);
        case 500: return launch_fft_xy_n<500, KIND>(h, map, nbatch, tw);
        case 512: return launch_fft_xy_n<512, KIND>(h, map, nbatch, tw);
        case 640: return launch_fft_xy_n<640, KIND>(h, map, nbatch, tw);
        case 768: return launch_fft_xy_n<768, KIND>(h, map, nbatch, tw);
        case 960: return launch_fft_xy_n<960, KIND>(h, map, nbatch, tw);
        case 1024: return launch_fft_xy_n<1024, KIND>(h, map, nbatch, tw);
        default: *handled = false; return DGPE_OK;
    }
}

// cuTensorMapEncodeTiled through the runtime (no link against libcuda)
static PFN_cuTensorMapEncodeTiled_v12000 tensor_map_encoder()
{
    static PFN_cuTensorMapEncodeTiled_v12000 fn = nullptr;
    static bool tried = false;
    if (!tried) {
        tried = true;
        void* p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
            q == cudaDriverEntryPointSuccess)
            fn = (PFN_cuTensorMapEncodeTiled_v12000)p;
        cudaGetLastError();
    }
    return fn;
}


// number of equal TMA boxes (<= 256 rows each) a line of n rows splits into; 0 if none
static constexpr int tma_boxes(int n)
{
    for (int k = (n + 255) / 256; k <= 8; ++k)
        if (n % k == 0 && n / k <= 256) return k;
    return 0;
}

// ---- K2 / K4 on the TMA pipeline (xyfft_tma.cuh): the long y lines ----
template <int N, bool INV, int NSTAGE>
static int launch_fft_tma_s(dgpe_handle* h)
{
    auto kern = k_fft_tma<N, INV, NSTAGE>;
    const size_t smem = (size_t)NSTAGE * N * TILE_COLS * sizeof(cplx) + 128;
    int rc = kernel_setup((const void*)kern, xy_threads<N>(), smem, nullptr);
    if (rc) return rc;
    const cuuint64_t nx = h->nx, ny = h->ny, nzh = h->nzh;
    constexpr int nbox = tma_boxes(N);
    static_assert(nbox > 0 && N % nbox == 0 && N / nbox <= 256, "line length must split into equal TMA boxes");
    cuuint64_t dims[3] = {2 * nzh, ny, nx}, strides[2] = {nzh * 16, ny * nzh * 16};
    cuuint32_t box[3] = {2 * TILE_COLS, (cuuint32_t)(N / nbox), 1}, estr[3] = {1, 1, 1};
    CUtensorMap tmap;
    CUresult cr = tensor_map_encoder()(&tmap, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 3, h->spec, dims, strides, box, estr,
                                       CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                                       CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (cr != CUDA_SUCCESS) return fail(DGPE_ERR_CUDA, "cuTensorMapEncodeTiled failed (%d)", (int)cr);
    TmaWalk W;
    W.n = N; W.box_rows = N / nbox;
    W.tiles_per_batch = (h->nzh + TILE_COLS - 1) / TILE_COLS;
    W.ntiles = W.tiles_per_batch * h->nx;
    kern<<<std::min(W.ntiles, h->num_sms), xy_threads<N>(), smem, h->stream>>>(tmap, W, h->tw_y);
    return check_launch("k_fft_tma");
}

template <int N>
static int launch_fft_tma_n(dgpe_handle* h, bool inverse)
{
    constexpr int NSTAGE = (3 * N * 128 <= 200 * 1024) ? 3 : 2;
    return inverse ? launch_fft_tma_s<N, true, NSTAGE>(h) : launch_fft_tma_s<N, false, NSTAGE>(h);
}

static int launch_fft_tma(dgpe_handle* h, bool inverse, bool* handled)
{
    *handled = h->use_tma_fft && tensor_map_encoder() != nullptr;
    if (!*handled) return DGPE_OK;
    switch (h->ny) {
        case 384: return launch_fft_tma_n<384>(h, inverse);
        case 480: return launch_fft_tma_n<480>(h, inverse);
        case 512: return launch_fft_tma_n<512>(h, inverse);
        case 640: return launch_fft_tma_n<640>(h, inverse);
        case 768: return launch_fft_tma_n<768>(h, inverse);
        default: *handled = false; return DGPE_OK;
    }
}

// ---- K3 on the TMA pipeline (xyfft_tma.cuh k_fft_tma_xudd): the long x lines ----
template <int N>
static int launch_fft_tma_xudd_n(dgpe_handle* h)
{
    constexpr int NSTAGE = (3 * N * 128 <= 200 * 1024) ? 3 : 2;
    auto kern = k_fft_tma_xudd<N, NSTAGE>;
    const size_t smem = (size_t)NSTAGE * N * TILE_COLS * sizeof(cplx) + 128;
    int rc = kernel_setup((const void*)kern, xy_threads<N>(), smem, nullptr);
    if (rc) return rc;
    const cuuint64_t nx = h->nx, ncols = (cuuint64_t)h->ny * h->nzh;
    constexpr int nbox = tma_boxes(N);
    static_assert(nbox > 0 && N % nbox == 0 && N / nbox <= 256, "line length must split into equal TMA boxes");
    cuuint64_t dims[3] = {2 * ncols, nx, 1}, strides[2] = {ncols * 16, nx * ncols * 16};
    cuuint32_t box[3] = {2 * TILE_COLS, (cuuint32_t)(N / nbox), 1}, estr[3] = {1, 1, 1};
    CUtensorMap tmap;
    CUresult cr = tensor_map_encoder()(&tmap, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 3, h->spec, dims, strides, box, estr,
                                       CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                                       CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (cr != CUDA_SUCCESS) return fail(DGPE_ERR_CUDA, "cuTensorMapEncodeTiled failed (%d)", (int)cr);
    TmaWalk W;
    W.n = N; W.box_rows = N / nbox;
    W.tiles_per_batch = (int)((ncols + TILE_COLS - 1) / TILE_COLS);
    W.ntiles = W.tiles_per_batch;
    UddArgs U{h->nzh, h->kx2, h->ky2, h->kz2, 2.0 * 3.14159265358979323846264338327950288 / ((double)h->nx * h->dx), h->inv_ntot, 0};
    kern<<<std::min(W.ntiles, h->num_sms), xy_threads<N>(), smem, h->stream>>>(tmap, W, h->tw_x, U, (int)ncols);
    return check_launch("k_fft_tma_xudd");
}

static int launch_fft_tma_xudd(dgpe_handle* h, bool* handled)
{
    *handled = (h->use_tma_k3 == 1 || (h->use_tma_k3 < 0 && h->nx >= 640)) && tensor_map_encoder() != nullptr;
    if (!*handled) return DGPE_OK;
    switch (h->nx) {
        case 384: return launch_fft_tma_xudd_n<384>(h);
        case 480: return launch_fft_tma_xudd_n<480>(h);
        case 512: return launch_fft_tma_xudd_n<512>(h);
        case 640: return launch_fft_tma_xudd_n<640>(h);
        case 768: return launch_fft_tma_xudd_n<768>(h);
        default: *handled = false; return DGPE_OK;
    }
}

// ---- K2 / K4 / K3 as k_fft_pair (xyfft_pair.cuh): two tiles per SM in different phases; N = 512.
//      (N = 768 would need 4-line tiles -- two teams of 8-line tiles are 1536 threads -- and TMA boxes with 64-byte rows
//      measured 5x slower: K2 0.81 -> 4.4 ms, K3 1.32 -> 6.4 ms at 768 x 768 x 384) ----
static bool fft_pair_wanted(const dgpe_handle* h, int n, bool xpass)
{
    if (n != 512 || !h->use_tma || h->force_generic || !tensor_map_encoder()) return false;
    if (h->opt.tma_pair == 0) return false;
    if (h->opt.tma_pair == 1) return true;
    return xpass ? DGPE_PAIR_DEFAULT_X : DGPE_PAIR_DEFAULT_Y;
}

template <int N, int KIND, int COLS, int NSTAGE>
static int launch_fft_pair(dgpe_handle* h)
{
    auto kern = k_fft_pair<N, KIND, COLS, NSTAGE>;
    constexpr int THREADS = 2 * pair_team_threads<N, COLS>();
    const size_t smem = (size_t)NSTAGE * N * COLS * sizeof(cplx) + 128;
    int rc = kernel_setup((const void*)kern, THREADS, smem, nullptr);
    if (rc) return rc;
    constexpr int nbox = tma_boxes(N);
    static_assert(nbox > 0 && N % nbox == 0 && N / nbox <= 256, "line length must split into equal TMA boxes");
    const cuuint64_t nx = h->nx, ny = h->ny, nzh = h->nzh, ncols = ny * nzh;
    cuuint64_t dims[3], strides[2];
    TmaWalk W;
    W.n = N; W.box_rows = N / nbox;
    if (KIND == FFT_X_UDD) {
        dims[0] = 2 * ncols; dims[1] = nx; dims[2] = 1; strides[0] = ncols * 16; strides[1] = nx * ncols * 16;
        W.tiles_per_batch = (int)((ncols + COLS - 1) / COLS);
        W.ntiles = W.tiles_per_batch;
    } else {
        dims[0] = 2 * nzh; dims[1] = ny; dims[2] = nx; strides[0] = nzh * 16; strides[1] = ny * nzh * 16;
        W.tiles_per_batch = (h->nzh + COLS - 1) / COLS;
        W.ntiles = W.tiles_per_batch * h->nx;
    }
    cuuint32_t box[3] = {2 * COLS, (cuuint32_t)(N / nbox), 1}, estr[3] = {1, 1, 1};
    CUtensorMap tmap;
    CUresult cr = tensor_map_encoder()(&tmap, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 3, h->spec, dims, strides, box, estr,
                                       CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                                       CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (cr != CUDA_SUCCESS) return fail(DGPE_ERR_CUDA, "cuTensorMapEncodeTiled failed (%d)", (int)cr);
    UddArgs U{h->nzh, h->kx2, h->ky2, h->kz2, 2.0 * 3.14159265358979323846264338327950288 / ((double)h->nx * h->dx), h->inv_ntot, 0};
    kern<<<std::min(W.ntiles, h->num_sms), THREADS, smem, h->stream>>>(tmap, W, KIND == FFT_X_UDD ? h->tw_x : h->tw_y, U, (int)ncols);
    return check_launch("k_fft_pair");
}

template <int KIND>
static int launch_fft_pair_n(dgpe_handle* h, int)
{
    return launch_fft_pair<512, KIND, 8, 3>(h);
}

static int launch_fft_y(dgpe_handle* h, bool inverse)
{
    const int nx = h->nx, ny = h->ny, nzh = h->nzh;
    LineMap my{ny, nzh, (long long)ny * nzh, 1, nzh};
    if (fft_pair_wanted(h, ny, false)) return inverse ? launch_fft_pair_n<FFT_INV>(h, ny) : launch_fft_pair_n<FFT_FWD>(h, ny);
    if (!h->force_generic) {
        bool handled = false;
        int rct = launch_fft_tma(h, inverse, &handled);
        if (rct || handled) return rct;
        int rc = inverse ? launch_fft_xy<FFT_INV>(h, ny, my, nx, h->tw_y, &handled)
                         : launch_fft_xy<FFT_FWD>(h, ny, my, nx, h->tw_y, &handled);
        if (rc || handled) return rc;
    }
    dim3 gy((nzh + 7) / 8, nx);
    const int ty = threads_for(h->plan_y.nbf);
    const size_t smy = sizeof(cplx) * TILE_COLS * (size_t)ny;
    int rcs;
    if (inverse) {
        if (ty <= 512) {
            if ((rcs = kernel_setup((const void*)k_fft_lines<true, 512>, ty, smy, nullptr))) return rcs;
            k_fft_lines<true, 512><<<gy, ty, smy, h->stream>>>(h->spec, my, h->plan_y);
        } else {
            if ((rcs = kernel_setup((const void*)k_fft_lines<true, 1024>, ty, smy, nullptr))) return rcs;
            k_fft_lines<true, 1024><<<gy, ty, smy, h->stream>>>(h->spec, my, h->plan_y);
        }
    } else {
        if (ty <= 512) {
            if ((rcs = kernel_setup((const void*)k_fft_lines<false, 512>, ty, smy, nullptr))) return rcs;
            k_fft_lines<false, 512><<<gy, ty, smy, h->stream>>>(h->spec, my, h->plan_y);
        } else {
            if ((rcs = kernel_setup((const void*)k_fft_lines<false, 1024>, ty, smy, nullptr))) return rcs;
            k_fft_lines<false, 1024><<<gy, ty, smy, h->stream>>>(h->spec, my, h->plan_y);
        }
    }
    return check_launch("k_fft_lines<y>");
}

static int launch_fft_x_udd(dgpe_handle* h)
{
    const int nx = h->nx, ny = h->ny, nzh = h->nzh;
    LineMap mx{nx, ny * nzh, 0, 1, (long long)ny * nzh};
    if (fft_pair_wanted(h, nx, true)) return launch_fft_pair_n<FFT_X_UDD>(h, nx);
    if (!h->force_generic) {
        bool handled = false;
        int rc = launch_fft_tma_xudd(h, &handled);
        if (rc || handled) return rc;
        rc = launch_fft_xy<FFT_X_UDD>(h, nx, mx, 1, h->tw_x, &handled);
        if (rc || handled) return rc;
    }
    const int tx = threads_for(h->plan_x.nbf);
    const size_t smx = sizeof(cplx) * TILE_COLS * (size_t)nx;
    int rcs;
    if (tx <= 512) {
        if ((rcs = kernel_setup((const void*)k_fft_x_udd<512>, tx, smx, nullptr))) return rcs;
        k_fft_x_udd<512><<<(ny * nzh + 7) / 8, tx, smx, h->stream>>>(h->spec, mx, h->plan_x, nzh, h->kx2, h->ky2, h->kz2,
                                                                     h->inv_ntot);
    } else {
        if ((rcs = kernel_setup((const void*)k_fft_x_udd<1024>, tx, smx, nullptr))) return rcs;
        k_fft_x_udd<1024><<<(ny * nzh + 7) / 8, tx, smx, h->stream>>>(h->spec, mx, h->plan_x, nzh, h->kx2, h->ky2, h->kz2,
                                                                      h->inv_ntot);
    }
    return check_launch("k_fft_x_udd");
}

// K1..K4: spec <- Udd~(k)/N * FFT(s2 |psi|^2), transformed back along x and y
static int launch_dipolar_spectrum(dgpe_handle* h, const cplx* psi)
{
    int rc;
    if ((rc = launch_k1(h, psi))) return rc;
    if ((rc = launch_fft_y(h, false))) return rc;
    if ((rc = launch_fft_x_udd(h))) return rc;
    return launch_fft_y(h, true);
}

// K5 in one of its modes
static int launch_c2r(dgpe_handle* h, cplx* psi, int kmode, double* out)
{
    if (h->zfast && kmode != 2) return launch_z_main(h, psi, kmode == 3 ? 3 : 0, out);
    const int nlines = h->nx * h->ny, M = h->nz / 2;
    NonlinArgs A;
    A.nlines = nlines; A.ny = h->ny; A.nz = h->nz;
    A.dt = h->dt; A.g = h->g; A.gdd = h->gdd;
    A.vx = h->vx; A.vy = h->vy; A.vz = h->vz;
    A.scal = h->scal; A.partials = h->partials; A.ticket = h->ticket; A.out = out;
    const int grid = (nlines + 7) / 8, thr = threads_for(h->plan_zh.nbf);
    const size_t sm = sizeof(cplx) * TILE_COLS * (size_t)(M + 1);
    auto go = [&](auto kern, auto* p) -> int {
        int rcs = kernel_setup((const void*)kern, thr, sm, nullptr);
        if (rcs) return rcs;
        kern<<<grid, thr, sm, h->stream>>>(p, h->spec, h->plan_zh, h->tw_split, A);
        return DGPE_OK;
    };
    int rcs;
    switch (kmode) {
        case 0: rcs = go(k_c2r_nonlin<0, cplx>, psi); break;
        case 1: rcs = go(k_c2r_nonlin<1, cplx>, psi); break;
        case 2: rcs = h->rpsi ? go(k_c2r_nonlin<2, double>, (double*)psi) : go(k_c2r_nonlin<2, cplx>, psi); break;
        default: rcs = go(k_c2r_nonlin<3, cplx>, psi); break;
    }
    if (rcs) return rcs;
    return check_launch("k_c2r_nonlin");
}

// ---- TMA-fed persistent sweep (xysweep_tma.cuh) ----
// can the TMA kernel take this sweep?  (whole tiles, a tile stage count >= 2 in shared memory, boxes <= 256 rows)
static bool tma_sweep_ok(const dgpe_handle* h, const LineMap& m, const AxisSweep& S, int* box_rows, int* nstage)
{
    if (!h->use_tma || h->force_generic || S.Lc != TMA_LC || S.G > 96 || m.ncols % TILE_COLS) return false;
    if (!tensor_map_encoder()) return false;
    const int nbox = tma_boxes(m.n);
    if (!nbox) return false;
    const size_t tile = (size_t)m.n * TILE_COLS * sizeof(cplx);
    int ns = (int)((200 * 1024) / tile);
    if (ns < 2) return false;
    // three stages when only one CTA fits on an SM anyway (tiles of 64 KB); two stages and several CTAs
    // per SM for the short lines, whose CTAs are small
    *nstage = (ns >= 3 && tile > 40 * 1024) ? 3 : 2;
    *box_rows = m.n / nbox;
    return true;
}

template <typename CT, bool CONSTTAB, int NSTAGE, int NTMAX>
static int launch_sweep_tma_s(dgpe_handle* h, cplx* psi, int axis, const LineMap& m, int box_rows, int thr,
                              const SweepTables<CT>& T, const SweepFold& F, const AxisSweep& S)
{
    auto kern = k_sweep_tma<CT, CONSTTAB, NSTAGE, NTMAX>;
    const size_t smem = (size_t)NSTAGE * m.n * TILE_COLS * sizeof(cplx) + 128;
    int ctas_per_sm = 1;
    int rc = kernel_setup((const void*)kern, thr, smem, &ctas_per_sm);
    if (rc) return rc;
    // psi viewed as doubles: x sweep {2 ny nz, nx, 1}, y sweep {2 nz, ny, nx}; box {16, box_rows, 1}
    const cuuint64_t nx = h->nx, ny = h->ny, nz = h->nzc;
    cuuint64_t dims[3], strides[2];
    if (axis == 0) { dims[0] = 2 * ny * nz; dims[1] = nx; dims[2] = 1; strides[0] = ny * nz * 16; strides[1] = nx * ny * nz * 16; }
    else { dims[0] = 2 * nz; dims[1] = ny; dims[2] = nx; strides[0] = nz * 16; strides[1] = ny * nz * 16; }
    cuuint32_t box[3] = {2 * TILE_COLS, (cuuint32_t)box_rows, 1}, estr[3] = {1, 1, 1};
    CUtensorMap tmap;
    CUresult cr = tensor_map_encoder()(&tmap, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 3, psi, dims, strides, box, estr,
                                       CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                                       CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (cr != CUDA_SUCCESS) return fail(DGPE_ERR_CUDA, "cuTensorMapEncodeTiled failed (%d)", (int)cr);
    TmaWalk W;
    W.n = m.n; W.box_rows = box_rows;
    W.tiles_per_batch = m.ncols / TILE_COLS;
    W.ntiles = W.tiles_per_batch * (axis == 0 ? 1 : h->nx);
    ChunkTabs<CT, TMA_LC> P;
    fill_chunk_tabs<CT, TMA_LC>(S, CONSTTAB, &P);
    const int grid = std::min(W.ntiles, h->num_sms * ctas_per_sm);
    kern<<<grid, thr, smem, h->stream>>>(tmap, W, T, F, P);
    return check_launch("k_sweep_tma");
}

template <typename CT, bool CONSTTAB>
static int launch_sweep_tma(dgpe_handle* h, cplx* psi, int axis, const LineMap& m, int box_rows, int nstage, int thr,
                            const SweepTables<CT>& T, const SweepFold& F, const AxisSweep& S)
{
    if (thr <= 256)
        return nstage == 2 ? launch_sweep_tma_s<CT, CONSTTAB, 2, 256>(h, psi, axis, m, box_rows, thr, T, F, S)
                           : launch_sweep_tma_s<CT, CONSTTAB, 3, 256>(h, psi, axis, m, box_rows, thr, T, F, S);
    if (thr <= 512)
        return nstage == 2 ? launch_sweep_tma_s<CT, CONSTTAB, 2, 512>(h, psi, axis, m, box_rows, thr, T, F, S)
                           : launch_sweep_tma_s<CT, CONSTTAB, 3, 512>(h, psi, axis, m, box_rows, thr, T, F, S);
    return nstage == 2 ? launch_sweep_tma_s<CT, CONSTTAB, 2, 768>(h, psi, axis, m, box_rows, thr, T, F, S)
                       : launch_sweep_tma_s<CT, CONSTTAB, 3, 768>(h, psi, axis, m, box_rows, thr, T, F, S);
}

template <typename CT, int LC, bool CONSTTAB, int NTMAX, int MINB>
static int launch_sweep_xy(dgpe_handle* h, cplx* psi, const LineMap& m, dim3 grid, int thr, const SweepTables<CT>& T,
                           const SweepFold& F, const AxisSweep& S)
{
    auto kern = k_sweep_xy<CT, LC, CONSTTAB, NTMAX, MINB>;
    ChunkTabs<CT, LC> P;
    fill_chunk_tabs<CT, LC>(S, CONSTTAB, &P);
    int ctas_per_sm = 0;
    int rc = kernel_setup((const void*)kern, thr, 0, &ctas_per_sm);
    if (rc) return rc;
    const int pf = (h->prefetch & (m.batch_stride ? PF_SWEEP_Y : PF_SWEEP_X)) ? h->pf_mult * ctas_per_sm * h->num_sms : 0;
    kern<<<grid, thr, 0, h->stream>>>(psi, m, T, F, pf, P);
    return check_launch("k_sweep_xy");
}

template <typename CT>
static int launch_sweep_t(dgpe_handle* h, cplx* psi, int axis, bool fold)
{
    const AxisSweep& S = h->sw[axis];
    const int nx = h->nx, ny = h->ny, nz = axis < 2 ? h->nzc : h->nz;      // x, y: complex columns along z
    SweepTables<CT> T;
    T.r = to_ct<CT>(S.r);
    T.omr2 = to_ct<CT>(1.0 - 2.0 * S.r);
    T.inv = (const CT*)S.inv; T.cc = (const CT*)S.cc; T.F = (const CT*)S.F; T.Gm = (const CT*)S.Gm;
    T.Ach = (const CT*)S.Ach; T.Bch = (const CT*)S.Bch; T.ztab = (const CT*)S.ztab;
    T.Lc = S.Lc; T.G = S.G; T.Kf = S.Kf; T.Kb = S.Kb; T.gU = S.gU;
    SweepFold F;
    F.enabled = fold ? 1 : 0;
    F.dV = h->dx * h->dy * h->dz;
    F.partials = h->partials; F.ticket = h->ticket; F.scal = h->scal;
    const int thr = threads_for(S.G);
    if (axis < 2 && !h->force_generic) {
        LineMap m = axis == 0 ? LineMap{nx, ny * nz, 0, 1, (long long)ny * nz} : LineMap{ny, nz, (long long)ny * nz, 1, nz};
        int box_rows = 0, nstage = 0;
        // Where the TMA pipeline pays (measured): the y axis from n = 384 up (512^3:
        // 0.75 vs 0.83 ms) and both axes for the long lines whose thread-loading CTAs are few and large
        // (768: 1.7 vs 2.3 ms).  On the x axis at n = 512 (rows ny*nz*16 bytes apart, one page each) it is
        // slower (0.94 vs 0.83 ms), and so it is for the short lines (256^3: 0.19 vs 0.11 ms).
        // Real-valued psi: the complex rows of the x axis are ny*nz*8 bytes apart, and there the TMA walk wins
        // on the x axis too (512^3: 0.39 vs 0.48 ms).
        const bool want_tma = (axis == 1 && m.n >= 384) || S.G > 64 || (h->use_tma_x) || (h->rpsi && m.n >= 384);
        if (want_tma && tma_sweep_ok(h, m, S, &box_rows, &nstage))
            return S.consttab ? launch_sweep_tma<CT, true>(h, psi, axis, m, box_rows, nstage, thr, T, F, S)
                              : launch_sweep_tma<CT, false>(h, psi, axis, m, box_rows, nstage, thr, T, F, S);
        dim3 grid((m.ncols + TILE_COLS - 1) / TILE_COLS, axis == 0 ? 1 : nx);
        if (S.Lc == 8 && S.G <= 64)
            return S.consttab ? launch_sweep_xy<CT, 8, true, 512, 2>(h, psi, m, grid, thr, T, F, S)
                              : launch_sweep_xy<CT, 8, false, 512, 2>(h, psi, m, grid, thr, T, F, S);
        if (S.Lc == 8 && S.G <= 96)
            return S.consttab ? launch_sweep_xy<CT, 8, true, 768, 1>(h, psi, m, grid, thr, T, F, S)
                              : launch_sweep_xy<CT, 8, false, 768, 1>(h, psi, m, grid, thr, T, F, S);
        if (S.Lc == 16 && S.G <= 64)
            return S.consttab ? launch_sweep_xy<CT, 16, true, 512, 1>(h, psi, m, grid, thr, T, F, S)
                              : launch_sweep_xy<CT, 16, false, 512, 1>(h, psi, m, grid, thr, T, F, S);
    }
    int rcs;
    if (axis == 0) {
        LineMap m{nx, ny * nz, 0, 1, (long long)ny * nz};
        const size_t sm = sweep_smem(nx, S.G, false);
        if ((rcs = kernel_setup((const void*)k_sweep<CT, false>, thr, sm, nullptr))) return rcs;
        k_sweep<CT, false><<<(ny * nz + 7) / 8, thr, sm, h->stream>>>(psi, m, T, F);
    } else if (axis == 1) {
        LineMap m{ny, nz, (long long)ny * nz, 1, nz};
        dim3 grid((nz + 7) / 8, nx);
        const size_t sm = sweep_smem(ny, S.G, false);
        if ((rcs = kernel_setup((const void*)k_sweep<CT, false>, thr, sm, nullptr))) return rcs;
        k_sweep<CT, false><<<grid, thr, sm, h->stream>>>(psi, m, T, F);
    } else {
        LineMap m{nz, nx * ny, 0, nz, 1};
        const size_t sm = sweep_smem(nz, S.G, true);
        if ((rcs = kernel_setup((const void*)k_sweep<CT, true>, thr, sm, nullptr))) return rcs;
        k_sweep<CT, true><<<(nx * ny + 7) / 8, thr, sm, h->stream>>>(psi, m, T, F);
    }
    return check_launch("k_sweep");
}

static int launch_sweep(dgpe_handle* h, cplx* psi, int axis, bool fold)
{
    if (axis == 2 && h->zfast && !fold) return launch_z_main(h, psi, 2, nullptr);
    return h->mode == DGPE_IMAG ? launch_sweep_t<double>(h, psi, axis, fold) : launch_sweep_t<cplx>(h, psi, axis, fold);
}

static int set_scal(dgpe_handle* h, int clear_bad)
{
    k_set_scal<<<1, 1, 0, h->stream>>>(h->scal, 1.0, 1.0, clear_bad);
    return check_launch("k_set_scal");
}

// One step = 8 kernels in the order of the method (K1..K5, sweeps x, y, z); 7 when the z-line kernels are
// available: the z sweep then runs fused into K5 and the sweeps go z, x, y (the three 1-D Cayley operators
// commute: R#26).  The norm is folded into the last sweep either way.  `mark` is called after each launch with the kernel index.
struct StepKernel { const char* name; double bytes; };

// the kernels of one step AS BUILT with their algorithmic bytes (each array read once and written once per pass)
static std::vector<StepKernel> step_kernels(const dgpe_handle* h)
{
    const double S = 16.0 * (double)h->nx * h->ny * h->nzh;
    const double N = (h->rpsi ? 0.5 : 1.0) * (double)h->N;      // in units of 16 bytes of psi
    std::vector<StepKernel> k;
    k.push_back({"K1 dens_r2c(z)", 16.0 * N + S});
    k.push_back({"K2 fft_y fwd", 2.0 * S});
    k.push_back({"K3 fft_x*Udd*ifft_x", 2.0 * S});
    k.push_back({"K4 fft_y inv", 2.0 * S});
    if (h->zfast) {
        k.push_back({"K5+K8 c2r(z)+nonlinear+sweep_z", S + 32.0 * N});     // the fused z sweep adds no traffic
        k.push_back({"K6 sweep_x", 32.0 * N});
        k.push_back({"K7 sweep_y(+norm)", 32.0 * N});
    } else {
        k.push_back({"K5 c2r(z)+nonlinear", S + 32.0 * N});
        k.push_back({"K6 sweep_x", 32.0 * N});
        k.push_back({"K7 sweep_y", 32.0 * N});
        k.push_back({"K8 sweep_z(+norm)", 32.0 * N});
    }
    return k;
}

template <typename Mark>
static int one_step(dgpe_handle* h, cplx* psi, Mark mark)
{
    const bool imag = h->mode == DGPE_IMAG;
    int rc, k = 0;
    if ((rc = launch_k1(h, psi))) return rc;
    mark(k++);
    if ((rc = launch_fft_y(h, false))) return rc;
    mark(k++);
    if ((rc = launch_fft_x_udd(h))) return rc;
    mark(k++);
    if ((rc = launch_fft_y(h, true))) return rc;
    mark(k++);
    if (h->zfast) {
        if ((rc = launch_z_main(h, psi, 1, nullptr))) return rc;
        mark(k++);
        if ((rc = launch_sweep(h, psi, 0, false))) return rc;
        mark(k++);
        if ((rc = launch_sweep(h, psi, 1, imag))) return rc;
        mark(k++);
        return DGPE_OK;
    }
    if ((rc = launch_c2r(h, psi, imag ? 0 : 1, nullptr))) return rc;
    mark(k++);
    if ((rc = launch_sweep(h, psi, 0, false))) return rc;
    mark(k++);
    if ((rc = launch_sweep(h, psi, 1, false))) return rc;
    mark(k++);
    if ((rc = launch_sweep(h, psi, 2, imag))) return rc;
    mark(k++);
    return DGPE_OK;
}

static int finish_steps(dgpe_handle* h, cplx* psi)
{
    int rc;
    k_scale<<<h->num_sms * 8, 256, 0, h->stream>>>(psi, h->rpsi ? h->N / 2 : h->N, h->scal);
    if ((rc = check_launch("k_scale"))) return rc;
    CU(cudaMemcpyAsync(h->h_out, h->scal, sizeof(double) * SC_COUNT, cudaMemcpyDeviceToHost, h->stream));
    return set_scal(h, 0);
}

static int check_finite(dgpe_handle* h)
{
    if (h->h_out[SC_BAD] != 0.0)
        return fail(DGPE_ERR_NONFINITE, "imaginary-time norm became zero or non-finite (last norm %g)", h->h_out[SC_NORM]);
    return DGPE_OK;
}

// nsteps steps on the handle's stream: the first ever step eagerly (it also finishes the lazy kernel
// attribute setup), the others as replays of the captured one-step graph.
static int run_steps(dgpe_handle* h, cplx* psi, int nsteps)
{
    int rc, s = 0;
    if (!h->warmed && nsteps > 0) {
        if ((rc = one_step(h, psi, [](int) {}))) return rc;
        h->warmed = true;
        s = 1;
    }
    if (h->use_graph && nsteps - s >= 2) {
        cudaGraphExec_t exec = nullptr;
        for (size_t i = 0; i < h->step_execs.size(); ++i)
            if (h->step_execs[i].first == psi) {
                std::rotate(h->step_execs.begin(), h->step_execs.begin() + i, h->step_execs.begin() + i + 1);
                exec = h->step_execs[0].second;
                break;
            }
        if (!exec) {
            if (!h->cap_stream) CU(cudaStreamCreateWithFlags(&h->cap_stream, cudaStreamNonBlocking));
            cudaStream_t user = h->stream;
            h->stream = h->cap_stream;
            cudaGraph_t graph = nullptr;
            cudaError_t e = cudaStreamBeginCapture(h->cap_stream, cudaStreamCaptureModeThreadLocal);
            rc = (e == cudaSuccess) ? one_step(h, psi, [](int) {}) : DGPE_ERR_CUDA;
            cudaError_t e2 = (e == cudaSuccess) ? cudaStreamEndCapture(h->cap_stream, &graph) : e;
            h->stream = user;
            if (rc || e2 != cudaSuccess || !graph) {
                if (graph) cudaGraphDestroy(graph);
                cudaGetLastError();
                return fail(DGPE_ERR_CUDA, "capturing the step graph failed: %s", cudaGetErrorString(e2));
            }
            e = cudaGraphInstantiate(&exec, graph, 0);
            cudaGraphDestroy(graph);
            if (e != cudaSuccess) return fail(DGPE_ERR_CUDA, "cudaGraphInstantiate failed: %s", cudaGetErrorString(e));
            if (h->step_execs.size() >= 4) {
                cudaGraphExecDestroy(h->step_execs.back().second);
                h->step_execs.pop_back();
            }
            h->step_execs.insert(h->step_execs.begin(), std::make_pair(psi, exec));
        }
        for (; s < nsteps; ++s) CU(cudaGraphLaunch(exec, h->stream));
        return DGPE_OK;
    }
    for (; s < nsteps; ++s)
        if ((rc = one_step(h, psi, [](int) {}))) return rc;
    return DGPE_OK;
}

extern "C" int dgpe_step(dgpe_handle* h, void* psi_, int nsteps)
{
    if (!h || !psi_) return fail(DGPE_ERR_ARG, "NULL handle or psi");
    { int rcd = check_device(h); if (rcd) return rcd; }
    if (nsteps < 0) return fail(DGPE_ERR_ARG, "nsteps = %d < 0", nsteps);
    if (nsteps == 0) return DGPE_OK;
    cplx* psi = (cplx*)psi_;
    int rc;
    if ((rc = set_scal(h, 1))) return rc;
    if ((rc = run_steps(h, psi, nsteps))) return rc;
    if (h->mode == DGPE_IMAG) {
        if ((rc = finish_steps(h, psi))) return rc;
        CU(cudaStreamSynchronize(h->stream));
        return check_finite(h);
    }
    return DGPE_OK;
}

extern "C" int dgpe_step_host(dgpe_handle* h, void* psi_host, int nsteps)
{
    if (!h || !psi_host) return fail(DGPE_ERR_ARG, "NULL handle or psi");
    { int rcd = check_device(h); if (rcd) return rcd; }
    if (nsteps < 0) return fail(DGPE_ERR_ARG, "nsteps = %d < 0", nsteps);
    const size_t bytes = (h->rpsi ? sizeof(double) : sizeof(cplx)) * (size_t)h->N;
    if (!h->psi_stage) {
        CU(cudaMalloc(&h->psi_stage, bytes));
        h->owned.push_back(h->psi_stage);
    }
    CU(cudaMemcpyAsync(h->psi_stage, psi_host, bytes, cudaMemcpyHostToDevice, h->stream));
    int rc;
    bool imag_done = false;
    if (nsteps > 0) {
        if ((rc = set_scal(h, 1))) return rc;
        if ((rc = run_steps(h, h->psi_stage, nsteps))) return rc;
        if (h->mode == DGPE_IMAG) {
            if ((rc = finish_steps(h, h->psi_stage))) return rc;
            imag_done = true;
        }
    }
    CU(cudaMemcpyAsync(psi_host, h->psi_stage, bytes, cudaMemcpyDeviceToHost, h->stream));
    CU(cudaStreamSynchronize(h->stream));
    return imag_done ? check_finite(h) : DGPE_OK;
}

extern "C" int dgpe_step_profile(dgpe_handle* h, void* psi_, int nsteps, double* ms)
{
    if (!h || !psi_ || !ms) return fail(DGPE_ERR_ARG, "NULL argument");
    { int rcd = check_device(h); if (rcd) return rcd; }
    if (nsteps < 1) return fail(DGPE_ERR_ARG, "nsteps = %d < 1", nsteps);
    const int NK = dgpe_launches_per_step(h);
    const size_t need = (size_t)nsteps * (NK + 1);
    while (h->prof_ev.size() < need) {
        cudaEvent_t e;
        CU(cudaEventCreate(&e));
        h->prof_ev.push_back(e);
    }
    cplx* psi = (cplx*)psi_;
    int rc;
    if ((rc = set_scal(h, 1))) return rc;
    for (int s = 0; s < nsteps; ++s) {
        cudaEvent_t* ev = &h->prof_ev[(size_t)s * (NK + 1)];
        cudaEventRecord(ev[0], h->stream);
        cudaStream_t st = h->stream;
        if ((rc = one_step(h, psi, [ev, st](int k) { cudaEventRecord(ev[k + 1], st); }))) return rc;
    }
    if (h->mode == DGPE_IMAG && (rc = finish_steps(h, psi))) return rc;
    CU(cudaStreamSynchronize(h->stream));
    for (int k = 0; k < NK; ++k) ms[k] = 0.0;
    for (int s = 0; s < nsteps; ++s) {
        cudaEvent_t* ev = &h->prof_ev[(size_t)s * (NK + 1)];
        for (int k = 0; k < NK; ++k) {
            float t = 0.f;
            CU(cudaEventElapsedTime(&t, ev[k], ev[k + 1]));
            ms[k] += (double)t / nsteps;
        }
    }
    return h->mode == DGPE_IMAG ? check_finite(h) : DGPE_OK;
}

extern "C" const char* dgpe_kernel_name(const dgpe_handle* h, int k)
{
    if (!h || k < 0 || k >= dgpe_launches_per_step(h)) return "";
    return step_kernels(h)[k].name;
}

// algorithmic bytes of kernel k AS BUILT: each array read once and written once per pass
extern "C" double dgpe_kernel_bytes(const dgpe_handle* h, int k)
{
    if (!h || k < 0 || k >= dgpe_launches_per_step(h)) return 0.0;
    return step_kernels(h)[k].bytes;
}

// ------------------------------------------------------------------------------------------------
// stage entry points
// ------------------------------------------------------------------------------------------------
extern "C" int dgpe_dipolar(dgpe_handle* h, const void* psi, void* phi)
{
    if (!h || !psi || !phi) return fail(DGPE_ERR_ARG, "NULL argument");
    { int rcd = check_device(h); if (rcd) return rcd; }
    int rc;
    if ((rc = launch_dipolar_spectrum(h, (const cplx*)psi))) return rc;
    return launch_c2r(h, const_cast<cplx*>((const cplx*)psi), 3, (double*)phi);
}

extern "C" int dgpe_nonlinear(dgpe_handle* h, void* psi)
{
    if (!h || !psi) return fail(DGPE_ERR_ARG, "NULL argument");
    { int rcd = check_device(h); if (rcd) return rcd; }
    int rc;
    if ((rc = launch_dipolar_spectrum(h, (const cplx*)psi))) return rc;
    return launch_c2r(h, (cplx*)psi, h->mode == DGPE_IMAG ? 0 : 1, nullptr);
}

extern "C" int dgpe_sweep(dgpe_handle* h, void* psi, int axis)
{
    if (!h || !psi) return fail(DGPE_ERR_ARG, "NULL argument");
    { int rcd = check_device(h); if (rcd) return rcd; }
    if (axis < 0 || axis > 2) return fail(DGPE_ERR_ARG, "axis %d not in 0..2", axis);
    return launch_sweep(h, (cplx*)psi, axis, false);
}

// ------------------------------------------------------------------------------------------------
// slab-decomposed step (SV section 8f NEXT-3): one rank's stages
// ------------------------------------------------------------------------------------------------
struct dgpe_slab {
    int P = 1, rank = 0, gnx = 0, gny = 0, nz = 0, nzh = 0, nxl = 0, nyl = 0;
    dgpe_handle* hx = nullptr;      // x slab [nxl][gny][nz]: whole lines along y and z
    dgpe_handle* hy = nullptr;      // y slab [gnx][nyl][nz]: whole lines along x (and z)
};

static dgpe_handle* make_view(int nx, int ny, int nz, int gnx, int gny, int x0, int y0, bool has_x, bool has_y,
                              double dx, double dy, double dz, double dt, double gamma, double nu, double lambda, double g,
                              double gdd, int mode, bool need_spec)
{
    dgpe_handle* h = new (std::nothrow) dgpe_handle();
    if (!h) { fail(DGPE_ERR_NOMEM, "host allocation failed"); return nullptr; }
    int* f = reinterpret_cast<int*>(&h->opt);
    for (size_t i = 0; i < sizeof(dgpe_options) / sizeof(int); ++i) f[i] = -1;
    h->nx = nx; h->ny = ny; h->nz = nz; h->nzh = nz / 2 + 1;
    h->gnx = gnx; h->gny = gny; h->x0 = x0; h->y0 = y0; h->has_x = has_x; h->has_y = has_y;
    h->rpsi = false; h->mode = mode; h->nzc = nz;
    h->dx = dx; h->dy = dy; h->dz = dz; h->dt = dt;
    h->gamma = gamma; h->nu = nu; h->lambda = lambda; h->g = g; h->gdd = gdd;
    h->N = (long long)nx * ny * nz;
    h->own_spec = need_spec;
    if (init_handle(h) != DGPE_OK) {
        char keep[sizeof(g_err)];
        std::memcpy(keep, g_err, sizeof(keep));
        dgpe_destroy(h);
        std::memcpy(g_err, keep, sizeof(keep));
        return nullptr;
    }
    return h;
}

extern "C" dgpe_slab* dgpe_slab_create(int nx, int ny, int nz, double dx, double dy, double dz, double dt, double gamma,
                                       double nu, double lambda, double g, double gdd, int mode, int nranks, int rank)
{
    g_err[0] = 0;
    g_err_code = DGPE_OK;
    auto bad = [](int code) -> dgpe_slab* { g_err_code = code; return nullptr; };
    const int ns[3] = {nx, ny, nz};
    for (int a = 0; a < 3; ++a) {
        if (ns[a] < 4) return bad(fail(DGPE_ERR_ARG, "grid size %d < 4", ns[a]));
        if (!smooth2357(ns[a])) return bad(fail(DGPE_ERR_ARG, "grid size %d is not of the form 2^a 3^b 5^c 7^d 11^e 13^f", ns[a]));
        if (ns[a] > DGPE_MAX_N) return bad(fail(DGPE_ERR_UNSUPPORTED, "grid size %d > %d", ns[a], DGPE_MAX_N));
    }
    if (nz % 2) return bad(fail(DGPE_ERR_ARG, "nz = %d must be even", nz));
    if (!(dx > 0.0) || !(dy > 0.0) || !(dz > 0.0) || !(dt > 0.0) || !std::isfinite(dx) || !std::isfinite(dy) ||
        !std::isfinite(dz) || !std::isfinite(dt))
        return bad(fail(DGPE_ERR_ARG, "dx, dy, dz, dt must be positive and finite"));
    if (mode != DGPE_IMAG && mode != DGPE_REAL) return bad(fail(DGPE_ERR_ARG, "mode %d is neither DGPE_IMAG nor DGPE_REAL", mode));
    // "NX and NY must be divisible by the number of processes ... programs will test ... and inform the user"
    if (nranks < 1 || rank < 0 || rank >= nranks) return bad(fail(DGPE_ERR_ARG, "rank %d of %d ranks", rank, nranks));
    if (nx % nranks || ny % nranks)
        return bad(fail(DGPE_ERR_ARG, "nx = %d and ny = %d must both be divisible by the number of ranks %d", nx, ny, nranks));
    dgpe_slab* s = new (std::nothrow) dgpe_slab();
    if (!s) return bad(fail(DGPE_ERR_NOMEM, "host allocation failed"));
    s->P = nranks; s->rank = rank; s->gnx = nx; s->gny = ny; s->nz = nz; s->nzh = nz / 2 + 1;
    s->nxl = nx / nranks; s->nyl = ny / nranks;
    s->hx = make_view(s->nxl, ny, nz, nx, ny, rank * s->nxl, 0, false, true, dx, dy, dz, dt, gamma, nu, lambda, g, gdd, mode, true);
    if (s->hx) s->hy = make_view(nx, s->nyl, nz, nx, ny, 0, rank * s->nyl, true, false, dx, dy, dz, dt, gamma, nu, lambda, g, gdd, mode, false);
    if (!s->hx || !s->hy) {
        char keep[sizeof(g_err)];
        std::memcpy(keep, g_err, sizeof(keep));
        dgpe_slab_destroy(s);
        std::memcpy(g_err, keep, sizeof(keep));
        return bad(DGPE_ERR_CUDA);
    }
    return s;
}

extern "C" void dgpe_slab_destroy(dgpe_slab* s)
{
    if (!s) return;
    dgpe_destroy(s->hx);
    dgpe_destroy(s->hy);
    delete s;
}

extern "C" int dgpe_slab_set_stream(dgpe_slab* s, void* cuda_stream)
{
    if (!s) return fail(DGPE_ERR_ARG, "NULL slab");
    s->hx->stream = s->hy->stream = (cudaStream_t)cuda_stream;
    return DGPE_OK;
}

extern "C" long long dgpe_slab_elems(const dgpe_slab* s, int spectrum)
{
    if (!s) return 0;
    return (long long)s->nxl * s->gny * (spectrum ? s->nzh : s->nz);
}

// block (q) of the slab array [nxl][gny][w] that belongs to rank q's y range, to / from a buffer [P][nxl][nyl][w]
// (the exchanged blocks are (NX/P) x (NY/P) x NZ each: P:L59; the strided side is what the paper's CUDA/MPI package maps
// with an MPI derived datatype, here one strided copy per peer)
static int slab_pack(const dgpe_slab* s, cudaStream_t st, const cplx* slab, cplx* buf, int w, bool unpack)
{
    const size_t width = (size_t)s->nyl * w * sizeof(cplx), pitch = (size_t)s->gny * w * sizeof(cplx);
    for (int q = 0; q < s->P; ++q) {
        const cplx* a = slab + (size_t)q * s->nyl * w;
        cplx* b = buf + (size_t)q * s->nxl * s->nyl * w;
        if (unpack) CU(cudaMemcpy2DAsync(const_cast<cplx*>(a), pitch, b, width, width, s->nxl, cudaMemcpyDeviceToDevice, st));
        else CU(cudaMemcpy2DAsync(b, width, a, pitch, width, s->nxl, cudaMemcpyDeviceToDevice, st));
    }
    return DGPE_OK;
}

extern "C" int dgpe_slab_begin(dgpe_slab* s)
{
    if (!s) return fail(DGPE_ERR_ARG, "NULL slab");
    int rc = check_device(s->hx);
    if (rc) return rc;
    if ((rc = set_scal(s->hx, 1))) return rc;
    return set_scal(s->hy, 1);
}

// a: density + R2C along z (K1) and FFT along y (K2) on the x slab; the half-spectrum leaves in blocks per peer
extern "C" int dgpe_slab_stage_a(dgpe_slab* s, const void* psi_x, void* spec_send)
{
    if (!s || !psi_x || !spec_send) return fail(DGPE_ERR_ARG, "NULL argument");
    int rc;
    if ((rc = launch_k1(s->hx, (const cplx*)psi_x))) return rc;
    if ((rc = launch_fft_y(s->hx, false))) return rc;
    return slab_pack(s, s->hx->stream, s->hx->spec, (cplx*)spec_send, s->nzh, false);
}

// b: FFT along x, Udd~(k)/N, inverse FFT along x (K3) in place on the y slab [nx][nyl][nzh] the exchange delivered
extern "C" int dgpe_slab_stage_b(dgpe_slab* s, void* spec_y)
{
    if (!s || !spec_y) return fail(DGPE_ERR_ARG, "NULL argument");
    cplx* own = s->hy->spec;
    s->hy->spec = (cplx*)spec_y;
    const int rc = launch_fft_x_udd(s->hy);
    s->hy->spec = own;
    return rc;
}

// c: the half-spectrum is back on the x slab: inverse FFT along y (K4), C2R along z + nonlinear exponential (K5),
//    sweeps along z and y; psi leaves in blocks per peer
extern "C" int dgpe_slab_stage_c(dgpe_slab* s, const void* spec_recv, void* psi_x, void* psi_send)
{
    if (!s || !spec_recv || !psi_x || !psi_send) return fail(DGPE_ERR_ARG, "NULL argument");
    dgpe_handle* h = s->hx;
    int rc;
    if ((rc = slab_pack(s, h->stream, h->spec, const_cast<cplx*>((const cplx*)spec_recv), s->nzh, true))) return rc;
    if ((rc = launch_fft_y(h, true))) return rc;
    if (h->zfast) {
        if ((rc = launch_z_main(h, (cplx*)psi_x, 1, nullptr))) return rc;
    } else {
        if ((rc = launch_c2r(h, (cplx*)psi_x, h->mode == DGPE_IMAG ? 0 : 1, nullptr))) return rc;
        if ((rc = launch_sweep(h, (cplx*)psi_x, 2, false))) return rc;
    }
    if ((rc = launch_sweep(h, (cplx*)psi_x, 1, false))) return rc;
    return slab_pack(s, h->stream, (const cplx*)psi_x, (cplx*)psi_send, s->nz, false);
}

// d: sweep along x in place on the y slab [nx][nyl][nz]; imaginary time: norm_part (DEVICE) <- this rank's sum |psi|^2 dV
extern "C" int dgpe_slab_stage_d(dgpe_slab* s, void* psi_y, double* norm_part)
{
    if (!s || !psi_y) return fail(DGPE_ERR_ARG, "NULL argument");
    dgpe_handle* h = s->hy;
    const bool imag = h->mode == DGPE_IMAG;
    if (imag && !norm_part) return fail(DGPE_ERR_ARG, "imaginary time needs norm_part");
    int rc;
    if ((rc = launch_sweep(h, (cplx*)psi_y, 0, imag))) return rc;
    if (imag) CU(cudaMemcpyAsync(norm_part, h->scal + SC_NORM, sizeof(double), cudaMemcpyDeviceToDevice, h->stream));
    return DGPE_OK;
}

// e: psi is back on the x slab; imaginary time: norm_total (DEVICE) = the sum of all ranks' norm_part -> the scale
//    factors of the next step's kernels
extern "C" int dgpe_slab_stage_e(dgpe_slab* s, const void* psi_recv, void* psi_x, const double* norm_total)
{
    if (!s || !psi_recv || !psi_x) return fail(DGPE_ERR_ARG, "NULL argument");
    dgpe_handle* h = s->hx;
    int rc;
    if ((rc = slab_pack(s, h->stream, (const cplx*)psi_x, const_cast<cplx*>((const cplx*)psi_recv), s->nz, true))) return rc;
    if (h->mode == DGPE_IMAG) {
        if (!norm_total) return fail(DGPE_ERR_ARG, "imaginary time needs norm_total");
        k_set_norm<<<1, 1, 0, h->stream>>>(h->scal, norm_total);
        if ((rc = check_launch("k_set_norm"))) return rc;
    }
    return DGPE_OK;
}

// end of a call of nsteps steps: imaginary time -> explicit rescale to unit norm, status of the norms seen
extern "C" int dgpe_slab_end(dgpe_slab* s, void* psi_x)
{
    if (!s || !psi_x) return fail(DGPE_ERR_ARG, "NULL argument");
    dgpe_handle* h = s->hx;
    if (h->mode != DGPE_IMAG) { CU(cudaStreamSynchronize(h->stream)); return DGPE_OK; }
    int rc;
    if ((rc = finish_steps(h, (cplx*)psi_x))) return rc;
    CU(cudaStreamSynchronize(h->stream));
    return check_finite(h);
}

// ------------------------------------------------------------------------------------------------
// observables
// ------------------------------------------------------------------------------------------------
static ObsArgs obs_args(dgpe_handle* h, double* out)
{
    ObsArgs A;
    A.nx = h->nx; A.ny = h->ny; A.nz = h->nz;
    A.x2 = h->x2; A.y2 = h->y2; A.z2 = h->z2;
    A.partials = h->partials; A.ticket = h->ticket; A.out = out;
    return A;
}

static int fetch(dgpe_handle* h, int count)
{
    CU(cudaMemcpyAsync(h->h_out, h->d_out, sizeof(double) * count, cudaMemcpyDeviceToHost, h->stream));
    CU(cudaStreamSynchronize(h->stream));
    return DGPE_OK;
}

static int moments(dgpe_handle* h, const void* psi)
{
    const int grid = std::min(h->nx * h->ny, h->num_sms * 8);
    if (h->rpsi) k_moments<double><<<grid, 256, 0, h->stream>>>((const double*)psi, obs_args(h, h->d_out));
    else k_moments<cplx><<<grid, 256, 0, h->stream>>>((const cplx*)psi, obs_args(h, h->d_out));
    int rc = check_launch("k_moments");
    if (rc) return rc;
    return fetch(h, 4);
}

extern "C" int dgpe_norm(dgpe_handle* h, const void* psi, double* norm)
{
    if (!h || !psi || !norm) return fail(DGPE_ERR_ARG, "NULL argument");
    { int rcd = check_device(h); if (rcd) return rcd; }
    int rc = moments(h, psi);
    if (rc) return rc;
    *norm = h->h_out[0] * h->dx * h->dy * h->dz;
    return DGPE_OK;
}

extern "C" int dgpe_rms(dgpe_handle* h, const void* psi, double rms[4])
{
    if (!h || !psi || !rms) return fail(DGPE_ERR_ARG, "NULL argument");
    { int rcd = check_device(h); if (rcd) return rcd; }
    int rc = moments(h, psi);
    if (rc) return rc;
    const double s = h->h_out[0];
    rms[0] = std::sqrt(h->h_out[1] / s);
    rms[1] = std::sqrt(h->h_out[2] / s);
    rms[2] = std::sqrt(h->h_out[3] / s);
    rms[3] = std::sqrt((h->h_out[1] + h->h_out[2] + h->h_out[3]) / s);
    return DGPE_OK;
}

extern "C" int dgpe_energy_terms(dgpe_handle* h, const void* psi_, double out[4])
{
    if (!h || !psi_ || !out) return fail(DGPE_ERR_ARG, "NULL argument");
    const void* psi = psi_;      // complex, or plain doubles in DGPE_IMAG_RPSI: every kernel below takes either
    int rc;
    if ((rc = check_device(h))) return rc;
    if ((rc = launch_dipolar_spectrum(h, (const cplx*)psi))) return rc;
    if ((rc = launch_c2r(h, const_cast<cplx*>((const cplx*)psi), 2, h->d_out))) return rc;
    const int grid = std::min(h->nx * h->ny, h->num_sms * 8);
    if (h->rpsi) k_kinetic<double><<<grid, 256, 0, h->stream>>>((const double*)psi, obs_args(h, h->d_out + 4));
    else k_kinetic<cplx><<<grid, 256, 0, h->stream>>>((const cplx*)psi, obs_args(h, h->d_out + 4));
    if ((rc = check_launch("k_kinetic"))) return rc;
    if ((rc = fetch(h, 8))) return rc;
    const double sV = h->h_out[0], sg = h->h_out[1], sdd = h->h_out[2], s = h->h_out[3];
    const double T = 0.5 * (h->h_out[4] / (h->dx * h->dx) + h->h_out[5] / (h->dy * h->dy) + h->h_out[6] / (h->dz * h->dz));
    out[0] = T / s;
    out[1] = sV / s;
    out[2] = h->g * sg / s;
    out[3] = h->gdd * sdd / s;
    return DGPE_OK;
}

extern "C" int dgpe_chempot(dgpe_handle* h, const void* psi, double* mu)
{
    if (!mu) return fail(DGPE_ERR_ARG, "NULL argument");
    double t[4];
    int rc = dgpe_energy_terms(h, psi, t);
    if (rc) return rc;
    *mu = t[0] + t[1] + t[2] + t[3];
    return DGPE_OK;
}

extern "C" int dgpe_energy(dgpe_handle* h, const void* psi, double* energy)
{
    if (!energy) return fail(DGPE_ERR_ARG, "NULL argument");
    double t[4];
    int rc = dgpe_energy_terms(h, psi, t);
    if (rc) return rc;
    *energy = t[0] + t[1] + 0.5 * t[2] + 0.5 * t[3];
    return DGPE_OK;
}

extern "C" double dgpe_bytes_per_step(const dgpe_handle* h)
{
    if (!h) return 0.0;
    const double N = (double)h->N, S = 16.0 * (double)h->nx * h->ny * h->nzh;
    // K1 16N+S, K2 2S, K3 2S, K4 2S, K5 S+32N, three sweeps 32N each (model M1);
    // real-valued psi: 8 bytes per point in every psi term, 72N + 8S (SV section 8f NEXT-2)
    return (h->rpsi ? 72.0 : 144.0) * N + 8.0 * S;
}

extern "C" int dgpe_launches_per_step(const dgpe_handle* h)
{
    return h ? (int)step_kernels(h).size() : 0;
}

// ------------------------------------------------------------------------------------------------
// dgpe_norm_noalloc -- the norm reduction for callers that cannot allocate (CUDA graph capture, tight
// serving loops, harnesses that forbid cudaMalloc).  Same two-stage deterministic reduction as the
// observables' k_moments (common.cuh grid_reduce: one partial per block, the last block adds them in a fixed
// order), but its scratch -- the partials and the arrival ticket, which dgpe_create takes from cudaMalloc --
// lives in ONE file-scope device array of fixed size, and the result goes to a DEVICE double of the caller.
// The entry point calls no cudaMalloc / cudaFree / allocating routine and does not synchronise.
//
// Every GPU that loads the library holds the array until the process exits (8448 bytes).  All calls share
// it and it keeps the last call's contents: the ticket is cleared on the caller's stream before every
// launch, the partials are overwritten before they are read.  Calls that OVERLAP on the GPU (two streams,
// two threads) race on it -- serialise them on one stream.
// ------------------------------------------------------------------------------------------------
static __device__ __align__(256) unsigned char g_noalloc_scratch[256 + 8 * DGPE_NOALLOC_MAX_NX];

// one block per x plane: partial[i] = sum over the plane of |psi|^2; out = dV * sum of the partials
__global__ void __launch_bounds__(256) k_norm_noalloc(const cplx* __restrict__ psi, long long plane, double dV,
                                                      double* __restrict__ partials, unsigned int* ticket,
                                                      double* __restrict__ out)
{
    __shared__ double red[32];
    const cplx* p = psi + (long long)blockIdx.x * plane;
    double acc[1] = {0.0};
    for (long long k = threadIdx.x; k < plane; k += blockDim.x) acc[0] += cabs2(p[k]);
    double tot[1];
    if (grid_reduce<1>(acc, partials, ticket, tot, red)) *out = tot[0] * dV;
}

// device address of the scratch array, looked up once per device with that device current (the array's
// name is a host-side stand-in in host code, not a device address)
static int noalloc_scratch(unsigned char** ptr)
{
    static std::mutex mu;
    static std::map<int, unsigned char*> by_device;
    int dev = -1;
    CU(cudaGetDevice(&dev));
    std::lock_guard<std::mutex> lock(mu);
    auto it = by_device.find(dev);
    if (it == by_device.end()) {
        unsigned char* p = nullptr;
        CU(cudaGetSymbolAddress((void**)&p, g_noalloc_scratch));
        if (!p) return fail(DGPE_ERR_CUDA, "cudaGetSymbolAddress returned a null scratch address");
        it = by_device.emplace(dev, p).first;
    }
    *ptr = it->second;
    return DGPE_OK;
}

extern "C" int dgpe_norm_noalloc(const void* psi, int nx, int ny, int nz, double dx, double dy, double dz,
                                 double* norm_device, void* cuda_stream)
{
    if (!psi || !norm_device) return fail(DGPE_ERR_ARG, "NULL argument");
    if (nx < 1 || ny < 1 || nz < 1) return fail(DGPE_ERR_ARG, "grid %d x %d x %d: every size must be >= 1", nx, ny, nz);
    if (nx > DGPE_NOALLOC_MAX_NX)
        return fail(DGPE_ERR_UNSUPPORTED, "dgpe_norm_noalloc: nx = %d exceeds DGPE_NOALLOC_MAX_NX = %d (one partial per x plane "
                                          "in the %d-byte static scratch array)", nx, DGPE_NOALLOC_MAX_NX, (int)sizeof(g_noalloc_scratch));
    if (!(dx > 0.0) || !(dy > 0.0) || !(dz > 0.0) || !std::isfinite(dx) || !std::isfinite(dy) || !std::isfinite(dz))
        return fail(DGPE_ERR_ARG, "dx, dy, dz must be positive and finite");
    unsigned char* scratch = nullptr;
    int rc = noalloc_scratch(&scratch);
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    unsigned int* ticket = reinterpret_cast<unsigned int*>(scratch);
    double* partials = reinterpret_cast<double*>(scratch + 256);
    CU(cudaMemsetAsync(ticket, 0, 256, st));             // the ticket must start at zero whatever the last call left
    k_norm_noalloc<<<nx, 256, 0, st>>>((const cplx*)psi, (long long)ny * nz, dx * dy * dz, partials, ticket, norm_device);
    return check_launch("k_norm_noalloc");
}
