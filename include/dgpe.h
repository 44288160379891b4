/*
 * dgpe.h -- C-ABI boundary of libdgpe: the split-step Crank-Nicolson (SSCN) time step of the
 * 3-D dipolar Gross-Pitaevskii equation on one NVIDIA B200 (sm_100a), complex fp64.
 *
 * Citations: P:Lnn = /root/reference/PAPER.md line nn (arXiv:1610.05329); BJ = BASELINE.json
 * (north_star, configs[i]); R#n = reading n of DESIGN.md section 3.
 *
 * The method ("Gross-Pitaevskii equation with contact and dipolar interaction in a harmonic
 * anisotropic trap"; "split-step Crank-Nicolson method ... imaginary or real time ... The
 * contribution of the dipolar interaction is evaluated by a Fourier transformation to momentum
 * space using a convolution theorem"; P:L39 real-to-complex transform of the density):
 *
 *   i dpsi/dt = [ -1/2 lap + 1/2 (gamma^2 x^2 + nu^2 y^2 + lambda^2 z^2) + g |psi|^2 + gdd Phi ] psi,
 *   Phi = Udd * |psi|^2,   Udd~(k) = (4 pi/3)(3 kz^2/|k|^2 - 1),  Udd~(0) = 0      (BJ:configs[0]),
 *   imaginary time: t -> -i tau, renormalised to  sum |psi|^2 dx dy dz = 1  after every step.
 *
 * One step (BJ:north_star (a)-(d)):
 *   (a) Phi = IFFT[ Udd~(k) FFT(|psi|^2) ];
 *   (b) psi <- exp(-i dt H) psi (real time) or exp(-dt H) psi (imaginary time), H = V + g|psi|^2 + gdd Phi;
 *   (c) three Crank-Nicolson line sweeps (x, y, z), Dirichlet psi = 0 on the end nodes of every axis;
 *   (d) imaginary time only: psi <- psi / sqrt(sum |psi|^2 dV).
 *
 * Layout: psi is complex double (re, im interleaved, 16 bytes per point), row-major
 * [nx][ny][nz], NX the slowest and NZ the contiguous dimension; x_i = (i - nx/2) dx (R#6).
 *
 * Memory: every `psi` argument is a DEVICE pointer to nx*ny*nz complex doubles, 16-byte aligned,
 * owned by the caller (e.g. a contiguous torch.complex128 CUDA tensor); the library never allocates
 * or frees it.  Every `double*` result argument is a HOST pointer.  The handle owns all device
 * workspace (half-spectrum buffer, per-axis tables, reduction scratch) and is immutable after
 * creation: a parameter quench is a second handle (BJ:configs[2]).
 *
 * Errors ("programs will test if these conditions are met, and inform the user"):
 * dgpe_create returns NULL, every other call returns a negative DGPE_ERR_* code, and
 * dgpe_last_error() returns a thread-local, human-readable description.  There is no CPU fallback.
 */
#ifndef DGPE_H
#define DGPE_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct dgpe_handle dgpe_handle;

/*
 * DGPE_IMAG_RPSI -- imaginary time with a REAL-VALUED wave function (the
 * paper's imaginary-time programs run ~1.65x faster than its real-time ones).  Every factor of the
 * imaginary-time step is real (exp(-dt H), the Crank-Nicolson matrices with r = dt/(4 d^2), the norm), so a
 * real psi stays real and the imaginary part of a complex psi carries nothing (R#5; the oracle's imaginary
 * part stays exactly 0 for real input: tests/test_oracle_pins.py).  In this mode every `psi` argument is
 * nx*ny*nz plain DOUBLES (8 bytes per point, same row-major layout, 16-byte aligned) and the step moves
 * 72N + 8S bytes instead of 144N + 8S.  The results equal those of DGPE_IMAG on the same psi with a zero
 * imaginary part.  nz must be one of the specialised z lengths (64, 128, 160, 192, 240, 250, 256, 320, 384,
 * 480, 500, 512, 640, 768), else dgpe_create fails with DGPE_ERR_UNSUPPORTED.  The observables take the same
 * doubles (their kernels are templated on the element type).
 */
enum { DGPE_IMAG = 0, DGPE_REAL = 1, DGPE_IMAG_RPSI = 2 };

enum {
    DGPE_OK = 0,
    DGPE_ERR_ARG = -1,       /* bad argument (see dgpe_create)                               */
    DGPE_ERR_CUDA = -2,      /* a CUDA runtime call or kernel launch failed                  */
    DGPE_ERR_NOMEM = -3,     /* host or device allocation failed                             */
    DGPE_ERR_UNSUPPORTED = -4, /* size outside what the kernels support                      */
    DGPE_ERR_NONFINITE = -5  /* imaginary time: the norm became 0, inf or NaN during the call */
};

/*
 * dgpe_create -- build a handle for one grid and one set of physical parameters.
 *   nx, ny, nz   grid points per axis; each >= 4, of the form 2^a 3^b 5^c 7^d 11^e 13^f (P:L130 FFT-friendly
 *                sizes), <= DGPE_MAX_N; nz even (the R2C half-spectrum, R#13).
 *   dx, dy, dz   grid spacings  (> 0);  dt  time step (> 0).
 *   gamma, nu, lambda   trap frequencies along x, y, z (R#2: gamma<->x slowest, lambda<->z).
 *   g, gdd       contact and dipolar interaction strengths; dipoles polarised along z (R#2).
 *   mode         DGPE_IMAG, DGPE_REAL or DGPE_IMAG_RPSI.
 * Returns NULL on error (DGPE_ERR_ARG / UNSUPPORTED / NOMEM / CUDA in dgpe_last_error()).
 * Uses the current CUDA device, which the handle remembers: every later call with this handle returns DGPE_ERR_ARG
 * if another device is current.  Allocates 16*nx*ny*(nz/2+1) bytes plus O(nx+ny+nz) tables.
 */
#define DGPE_MAX_N 1024
dgpe_handle* dgpe_create(int nx, int ny, int nz, double dx, double dy, double dz, double dt,
                         double gamma, double nu, double lambda, double g, double gdd, int mode);

/*
 * dgpe_create_ex -- dgpe_create with kernel-selection options, for A/B measurements and for the in-repo
 * cross-checks of one kernel family against another (tests/test_gpu_parity.py test_kernel_variants_agree).
 * Every field: -1 = the library's default (what dgpe_create uses; opt = NULL means all defaults).  The results
 * are the same within rounding whatever the options; the library itself never reads the environment.
 */
typedef struct dgpe_options {
    int generic;      /* 1: the runtime-plan (generic) kernels everywhere                                   */
    int tma;          /* 0: x/y sweeps load and store through the threads; 2: TMA on the x axis as well     */
    int tma_fft;      /* 0: K2/K4 through the threads (k_fft_xy) instead of the TMA pipeline                 */
    int tma_k3;       /* 0 | 1: K3 never | always on the TMA pipeline (default: from nx = 640 up)           */
    int graph;        /* 0: plain launches instead of replaying the captured one-step CUDA graph            */
    int prefetch;     /* mask of kernel families with the L2 prefetch of the next residency:
                         1 z lines, 2 y sweep, 4 x sweep, 8 y FFT, 16 x FFT                                 */
    int pf_mult;      /* prefetch distance in units of one residency (default 1)                            */
    int tma_pair;     /* 0 | 1: never | always run K2, K3, K4 at nx, ny = 512 as k_fft_pair (two tiles per SM in different
                         phases on the TMA pipeline); default: K3 only                                        */
    int reserved[8];  /* set to -1 */
} dgpe_options;
dgpe_handle* dgpe_create_ex(int nx, int ny, int nz, double dx, double dy, double dz, double dt,
                            double gamma, double nu, double lambda, double g, double gdd, int mode,
                            const dgpe_options* opt);

/* The DGPE_ERR_* code of this thread's last failed dgpe_create / dgpe_create_ex (DGPE_OK if it succeeded). */
int dgpe_last_error_code(void);

/* Frees the handle's device and host memory.  NULL is allowed. */
void dgpe_destroy(dgpe_handle* h);

/* All later work of this handle is enqueued on `cuda_stream` (a cudaStream_t passed as void*;
   NULL = the legacy default stream, which is also the initial setting). */
int dgpe_set_stream(dgpe_handle* h, void* cuda_stream);

/*
 * dgpe_step -- advance psi in place by nsteps full SSCN steps (BJ:north_star (a)-(d)).
 * All kernels are enqueued on the handle's stream without host synchronisation inside the loop.
 * Imaginary time: the per-step renormalisation (d) is carried as a scalar into the next step's
 * kernels and applied explicitly once at the end, so psi has unit norm on return; the call then
 * waits for the stream and returns DGPE_ERR_NONFINITE if a norm was 0/inf/NaN (R#18: no clamp).
 * Real time: psi is never rescaled; the call returns after enqueueing.
 * nsteps = 0 is a no-op.  Errors: DGPE_ERR_ARG (NULL, nsteps < 0), DGPE_ERR_CUDA.
 */
int dgpe_step(dgpe_handle* h, void* psi, int nsteps);

/* Observables (R#14-R#17).  Each call enqueues on the handle's stream, waits for it and writes HOST
   doubles.  psi need not be normalised; mu, E and rms are divided by the norm.
     norm   = sum |psi|^2 dx dy dz                               (the integral, not its root)
     mu     = [T + sum(V n + g n^2 + gdd Phi n) dV] / norm
     energy = [T + sum(V n + g n^2/2 + gdd Phi n/2) dV] / norm
     T      = sum_axes 1/2 sum_links |psi_{j+1} - psi_j|^2 / d^2 dV,  links j = -1..n-1, psi_-1 = psi_n = 0
     rms    = { sqrt<x^2>, sqrt<y^2>, sqrt<z^2>, sqrt<x^2+y^2+z^2> }  about the origin            */
int dgpe_norm(dgpe_handle* h, const void* psi, double* norm);
int dgpe_chempot(dgpe_handle* h, const void* psi, double* mu);
int dgpe_energy(dgpe_handle* h, const void* psi, double* energy);
int dgpe_rms(dgpe_handle* h, const void* psi, double rms[4]);
/* out[0] = T, out[1] = <V>, out[2] = g<n>, out[3] = gdd<Phi>, each divided by the norm
   (mu = sum of the four; energy = out0 + out1 + out2/2 + out3/2). */
int dgpe_energy_terms(dgpe_handle* h, const void* psi, double out[4]);

/* Stage entry points (diagnostics and per-stage parity tests; same kernels as dgpe_step):
     dgpe_dipolar    phi (DEVICE, nx*ny*nz doubles) <- Phi of step (a) for the given psi
     dgpe_nonlinear  psi <- steps (a)+(b) only
     dgpe_sweep      psi <- one Crank-Nicolson sweep of step (c) along axis 0 = x, 1 = y, 2 = z   */
int dgpe_dipolar(dgpe_handle* h, const void* psi, void* phi);
int dgpe_nonlinear(dgpe_handle* h, void* psi);
int dgpe_sweep(dgpe_handle* h, void* psi, int axis);

/*
 * dgpe_step_host -- the same as dgpe_step for a wave function in HOST memory: copies nx*ny*nz complex
 * doubles from psi_host (pinned memory makes the copies asynchronous DMA; pageable memory works, slower)
 * to a device buffer the handle owns (allocated on first use, 16*nx*ny*nz bytes), runs nsteps steps,
 * copies the result back into psi_host and waits for the stream.  Same return codes as dgpe_step,
 * plus DGPE_ERR_NOMEM if the staging buffer cannot be allocated.
 */
int dgpe_step_host(dgpe_handle* h, void* psi_host, int nsteps);

/*
 * dgpe_step_profile -- run nsteps steps exactly as dgpe_step does, with a CUDA event recorded on the
 * handle's stream between consecutive kernels; ms[k] (HOST, dgpe_launches_per_step() doubles) receives
 * the average duration in milliseconds of kernel k of the step.  Waits for the stream.
 * dgpe_kernel_name(k) / dgpe_kernel_bytes(h, k) give the name and the algorithmic bytes of kernel k.
 */
int dgpe_step_profile(dgpe_handle* h, void* psi, int nsteps, double* ms);
const char* dgpe_kernel_name(const dgpe_handle* h, int k);
double dgpe_kernel_bytes(const dgpe_handle* h, int k);

/* Waits for the handle's stream. */
int dgpe_synchronize(dgpe_handle* h);

/* Algorithmic bytes one step moves (model of the kernels as built) and the
   number of kernel launches per step; used by bench.py for the roofline line. */
double dgpe_bytes_per_step(const dgpe_handle* h);
int dgpe_launches_per_step(const dgpe_handle* h);

/*
 * Slab-decomposed step -- one rank's share of a step distributed over `nranks` GPUs.
 * The paper distributes the data "along NX": rank p owns the x slab psi[p NX/P .. (p+1) NX/P)[NY][NZ], whole
 * lines along y and z, so the y and z passes and sweeps are local; "anything needing the whole NX extent" --
 * the x pass of the dipolar convolution and the x sweep -- runs after an all-to-all exchange that leaves the data
 * "locally transposed" as NX x (NY/P) x NZ, each rank sending every peer one (NX/P) x (NY/P) x NZ block,
 * and is followed by the exchange back.  The library does the local stages and the strided packing of the blocks; the
 * exchanges themselves belong to the caller (torch.distributed over NCCL in paper_1610_05329_b200/sharded.py, or local
 * copies when all ranks are emulated on one device), which is why every buffer below is caller-owned:
 *
 *   begin
 *   a(psi_x, spec_send)               K1, K2; spec_send[q] = block for rank q            -> all-to-all -> spec_y
 *   b(spec_y)                         K3 in place on [NX][NY/P][NZ/2+1]                   -> all-to-all back -> spec_recv
 *   c(spec_recv, psi_x, psi_send)     K4, K5 (+ z sweep), y sweep; psi_send[q] = block q  -> all-to-all -> psi_y
 *   d(psi_y, norm_part)               x sweep in place on [NX][NY/P][NZ]; norm_part = own part of the norm
 *                                                              -> all-to-all back -> psi_recv; all-reduce(norm_part) -> norm_total
 *   e(psi_recv, psi_x, norm_total)    psi back in the x slab; scale factors of the next step
 *   ... nsteps times ...; end(psi_x)  imaginary time: explicit rescale, DGPE_ERR_NONFINITE if a norm was 0/inf/NaN
 *
 * A buffer of blocks is [P][NX/P][NY/P][w] complex doubles (w = NZ/2+1 for the half-spectrum, NZ for psi); received from
 * all ranks in rank order it IS the y slab [NX][NY/P][w], and the y slab is the send buffer of the way back.
 * dgpe_slab_elems(s, spectrum) = (NX/P) NY w: the element count of every one of these buffers.
 * Every pointer is a DEVICE pointer; all work is enqueued on the slab's stream; sweeps run in the order z, y, x (R#26).
 * Errors as dgpe_create / dgpe_step; NX and NY must be divisible by nranks.  DGPE_IMAG and DGPE_REAL only.
 */
typedef struct dgpe_slab dgpe_slab;
dgpe_slab* dgpe_slab_create(int nx, int ny, int nz, double dx, double dy, double dz, double dt, double gamma, double nu,
                            double lambda, double g, double gdd, int mode, int nranks, int rank);
void dgpe_slab_destroy(dgpe_slab* s);
int dgpe_slab_set_stream(dgpe_slab* s, void* cuda_stream);
long long dgpe_slab_elems(const dgpe_slab* s, int spectrum);
int dgpe_slab_begin(dgpe_slab* s);
int dgpe_slab_stage_a(dgpe_slab* s, const void* psi_x, void* spec_send);
int dgpe_slab_stage_b(dgpe_slab* s, void* spec_y);
int dgpe_slab_stage_c(dgpe_slab* s, const void* spec_recv, void* psi_x, void* psi_send);
int dgpe_slab_stage_d(dgpe_slab* s, void* psi_y, double* norm_part);
int dgpe_slab_stage_e(dgpe_slab* s, const void* psi_recv, void* psi_x, const double* norm_total);
int dgpe_slab_end(dgpe_slab* s, void* psi_x);

/*
 * dgpe_norm_noalloc -- norm = sum |psi|^2 dx dy dz (BJ:north_star (d); R#14, R#15) WITHOUT any allocation, for callers
 * that cannot call cudaMalloc: code under CUDA graph capture, tight serving loops, harnesses that forbid it.  No handle:
 *   psi          DEVICE, nx*ny*nz complex doubles, row-major [nx][ny][nz] (as everywhere in this header)
 *   norm_device  DEVICE, one double the caller owns; written asynchronously on `cuda_stream` (cudaStream_t as void*,
 *                NULL = legacy default stream).  The call does not synchronise and copies nothing to the host.
 * The scratch of the reduction (one partial per x plane and an arrival ticket) is a static device array of
 * 256 + 8*DGPE_NOALLOC_MAX_NX = 8448 bytes that every GPU loading the library holds until exit; nx beyond
 * DGPE_NOALLOC_MAX_NX is rejected with DGPE_ERR_UNSUPPORTED.  All calls share that array and it keeps the last call's
 * contents (the call clears what must start at zero): calls that OVERLAP on the GPU -- different streams or threads --
 * race on it; issue them on one stream.  Uses the current CUDA device, which must hold psi and norm_device.
 * Deterministic (fixed summation order); equals dgpe_norm to rounding (another summation order).
 * Errors: DGPE_ERR_ARG (NULL, sizes < 1, spacings), DGPE_ERR_UNSUPPORTED (nx too large), DGPE_ERR_CUDA.
 */
#define DGPE_NOALLOC_MAX_NX 1024
int dgpe_norm_noalloc(const void* psi, int nx, int ny, int nz, double dx, double dy, double dz,
                      double* norm_device, void* cuda_stream);

/* Thread-local description of the last error ("" if none). Never NULL. */
const char* dgpe_last_error(void);

#ifdef __cplusplus
}
#endif
#endif
