/*
 * dgpe_oracle.h -- CPU ORACLE for the 3-D dipolar Gross-Pitaevskii split-step
 * Crank-Nicolson (SSCN) time step.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may load it.  It shares no code,
 * header, table or constant generator with the CUDA library in
 * paper_1610_05329_b200/csrc (whose boundary is include/dgpe.h).
 *
 * Plain C99, single thread, fp64 throughout, no blocking / fusion / reordering beyond
 * what the algorithm states.  Citations:  P:Lnn = /root/reference/PAPER.md line nn;
 * BJ = BASELINE.json (north_star / configs[i]);  R#n = reading n in DESIGN.md section 3
 * (= SURVEY.md section 8(c) item n).
 *
 * What it computes (one call of odgpe_step does nsteps of):
 *   1. n = |psi|^2                                              (BJ:north_star (a))
 *   2. Phi = IDFT3[ Udd(k) * DFT3(n) ] / (nx ny nz)             ("convolution theorem";
 *      Udd(k) = (4 pi/3)(3 kz^2/|k|^2 - 1), Udd(0) = 0           BJ:configs[0])
 *   3. psi <- exp(-dt H) psi  (imag)  or  exp(-i dt H) psi (real),
 *      H = (gamma^2 x^2 + nu^2 y^2 + lambda^2 z^2)/2 + g n + gdd Phi   (BJ:north_star (b))
 *   4. Crank-Nicolson sweep along x, then y, then z (Thomas)     (BJ:north_star (c))
 *   5. imag only: psi <- psi / sqrt(dV * sum |psi|^2)            (BJ:north_star (d))
 *
 * Pins (tests/test_oracle_pins.py, all -m "not gpu"):
 *   odgpe_dft1 / odgpe_dft3 ...... brute-force O(n^2) DFT, radix 2, 3 and mixed sizes     (P1, P2)
 *   odgpe_dipolar ................ plane-wave closed form, cubic-symmetry zero, Gaussian
 *                                  closed form, numpy.fft on random densities            (P3-P6)
 *   odgpe_sweep .................. dense Gaussian elimination on tiny lines, real and
 *                                  imaginary r                                            (P7)
 *   odgpe_nonlinear .............. closed form with g = gdd = 0; numpy expression        (P3b)
 *   odgpe_step (real) ............ norm conservation <= 1e-12 per step                    (P8)
 *   odgpe_norm/rms/chempot/energy  Gaussian closed forms                                  (P9)
 *   odgpe_step (imag, g=gdd=0) ... separable dense eigen-solution of the 1-D step map     (P10-P12)
 *   odgpe_step (imag, full) ...... dense-matrix restatement on tiny grids; third-
 *                                  implementation values of SURVEY 8(c) P13               (P13)
 *   real-time step with interactions beyond P8 + the tiny-grid dense restatement:
 *   no closed form exists -- see DESIGN.md section 4.
 */
#ifndef DGPE_ORACLE_H
#define DGPE_ORACLE_H

#include <complex.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct odgpe_handle odgpe_handle;

enum { ODGPE_IMAG = 0, ODGPE_REAL = 1 };
enum {
    ODGPE_OK = 0,
    ODGPE_ERR_ARG = -1,
    ODGPE_ERR_NOMEM = -3,
    ODGPE_ERR_NONFINITE = -5
};

/* psi: host pointer, complex double, row-major [nx][ny][nz], z contiguous. */
odgpe_handle *odgpe_create(int nx, int ny, int nz, double dx, double dy, double dz, double dt,
                           double gamma, double nu, double lambda, double g, double gdd, int mode);
void odgpe_destroy(odgpe_handle *h);

int odgpe_step(odgpe_handle *h, double complex *psi, int nsteps);
int odgpe_norm(odgpe_handle *h, const double complex *psi, double *norm);
int odgpe_chempot(odgpe_handle *h, const double complex *psi, double *mu);
int odgpe_energy(odgpe_handle *h, const double complex *psi, double *energy);
int odgpe_rms(odgpe_handle *h, const double complex *psi, double rms[4]);

/* ---- stage entry points (what the pins and the per-stage parity tests call) ---- */
/* unnormalised DFT of one contiguous line, sign = -1 forward (e^{-i k x}), +1 inverse */
int odgpe_dft1(int n, double complex *line, int sign);
/* unnormalised 3-D DFT in place on [nx][ny][nz] */
int odgpe_dft3(int nx, int ny, int nz, double complex *a, int sign);
/* Phi from a real density (step 2) */
int odgpe_dipolar(odgpe_handle *h, const double *dens, double *phi);
/* step 1-3 only */
int odgpe_nonlinear(odgpe_handle *h, double complex *psi);
/* step 4 for one axis (0 = x, 1 = y, 2 = z) */
int odgpe_sweep(odgpe_handle *h, double complex *psi, int axis);
/* components of the energy functional, each divided by norm:
   out[0] = T, out[1] = <V>, out[2] = g <n>, out[3] = gdd <Phi>  (so mu = T+V+out2+out3) */
int odgpe_energy_terms(odgpe_handle *h, const double complex *psi, double out[4]);

#ifdef __cplusplus
}
#endif
#endif
