/*
 * dgpe_oracle.c -- CPU ORACLE (test infrastructure, NOT the product; see dgpe_oracle.h).
 *
 * Plain, slow, single-threaded C99 statement of the split-step Crank-Nicolson step of the
 * 3-D dipolar Gross-Pitaevskii equation, in the order and notation of DESIGN.md section 2
 * (BJ:north_star (a)-(d); BJ:configs[0]).  It has its own
 * mixed-radix FFT (the DFT definition applied recursively by prime factor) and its own
 * Thomas solver, and shares nothing with the CUDA path.
 */
#include "dgpe_oracle.h"

#include <math.h>
#include <stdlib.h>
#include <string.h>

typedef double complex cplx;

struct odgpe_handle {
    int nx, ny, nz;
    double dx, dy, dz, dt;
    double gamma, nu, lambda, g, gdd;
    int mode;
    /* Thomas tables per axis (R#9): inv_j and c_j for unknowns j = 1..n-2 */
    cplx r[3];
    cplx *inv[3];
    cplx *c[3];
};

static const double ODGPE_PI = 3.14159265358979323846264338327950288;

/* ------------------------------------------------------------------------------------ */
/* FFT: the DFT definition, split recursively by the smallest prime factor p of n        */
/*   X_k = sum_j x_j w_n^{jk},  j = p*j' + q  =>                                         */
/*   X_{k + m*s} = sum_q w_n^{q k} w_p^{q s} * [DFT_m of the q-th decimated sequence]_k  */
/* with m = n/p, k = 0..m-1, s = 0..p-1.  Radix 2 and 3 are the cases the configs need   */
/* (BJ:configs[4]); any other prime p falls through the same O(p^2) butterfly.   */
/* ------------------------------------------------------------------------------------ */

static int smallest_factor(int n)
{
    for (int p = 2; p * p <= n; ++p)
        if (n % p == 0) return p;
    return n;
}

/* w holds exp(sign*2*pi*i*j/N) for j = 0..N-1; this level has length n = N/wstep */
static void dft_rec(int n, const cplx *in, int istride, cplx *out, const cplx *w, int N, int wstep,
                    cplx *tmp)
{
    if (n == 1) {
        out[0] = in[0];
        return;
    }
    int p = smallest_factor(n);
    int m = n / p;
    for (int q = 0; q < p; ++q)
        dft_rec(m, in + (size_t)q * istride, istride * p, out + (size_t)q * m, w, N, wstep * p, tmp);
    for (int k = 0; k < m; ++k) {
        for (int q = 0; q < p; ++q) {
            long idx = ((long)q * k * wstep) % N;              /* w_n^{qk} */
            tmp[q] = out[(size_t)q * m + k] * w[idx];
        }
        for (int s = 0; s < p; ++s) {
            cplx acc = 0.0;
            for (int q = 0; q < p; ++q) {
                long idx = ((long)q * s * m * wstep) % N;      /* w_p^{qs} = w_n^{q s m} */
                acc += tmp[q] * w[idx];
            }
            out[(size_t)s * m + k] = acc;                       /* safe: reads of column k done */
        }
    }
}

typedef struct {
    int n;
    int sign;
    cplx *w;     /* n twiddles */
    cplx *buf;   /* n */
    cplx *tmp;   /* n (>= largest prime factor) */
} dft_plan;

static int plan_init(dft_plan *pl, int n, int sign)
{
    pl->n = n;
    pl->sign = sign;
    pl->w = (cplx *)malloc(sizeof(cplx) * (size_t)n);
    pl->buf = (cplx *)malloc(sizeof(cplx) * (size_t)n);
    pl->tmp = (cplx *)malloc(sizeof(cplx) * (size_t)n);
    if (!pl->w || !pl->buf || !pl->tmp) return ODGPE_ERR_NOMEM;
    for (int j = 0; j < n; ++j) {
        double a = 2.0 * ODGPE_PI * (double)j / (double)n;
        pl->w[j] = cos(a) + (double)sign * sin(a) * I;
    }
    return ODGPE_OK;
}

static void plan_free(dft_plan *pl)
{
    free(pl->w);
    free(pl->buf);
    free(pl->tmp);
    pl->w = pl->buf = pl->tmp = NULL;
}

/* transform n elements at a + j*stride in place */
static void plan_exec(dft_plan *pl, cplx *a, size_t stride)
{
    int n = pl->n;
    /* dft_rec reads "in" with a stride and writes "out" contiguously */
    dft_rec(n, a, (int)stride, pl->buf, pl->w, n, 1, pl->tmp);
    for (int j = 0; j < n; ++j) a[(size_t)j * stride] = pl->buf[j];
}

int odgpe_dft1(int n, double complex *line, int sign)
{
    if (n < 1 || !line || (sign != 1 && sign != -1)) return ODGPE_ERR_ARG;
    dft_plan pl;
    int rc = plan_init(&pl, n, sign);
    if (rc == ODGPE_OK) plan_exec(&pl, line, 1);
    plan_free(&pl);
    return rc;
}

int odgpe_dft3(int nx, int ny, int nz, double complex *a, int sign)
{
    if (nx < 1 || ny < 1 || nz < 1 || !a || (sign != 1 && sign != -1)) return ODGPE_ERR_ARG;
    /* strides are passed as int to dft_rec: the deepest level uses stride * n */
    if ((double)nx * ny * nz >= 2147483647.0) return ODGPE_ERR_ARG;
    dft_plan px, py, pz;
    int rc = plan_init(&pz, nz, sign);
    if (rc == ODGPE_OK) rc = plan_init(&py, ny, sign);
    else { plan_free(&pz); return rc; }
    if (rc == ODGPE_OK) rc = plan_init(&px, nx, sign);
    else { plan_free(&pz); plan_free(&py); return rc; }
    if (rc != ODGPE_OK) { plan_free(&pz); plan_free(&py); plan_free(&px); return rc; }

    size_t sy = (size_t)nz, sx = (size_t)ny * nz;
    for (int i = 0; i < nx; ++i)
        for (int j = 0; j < ny; ++j) plan_exec(&pz, a + i * sx + j * sy, 1);
    for (int i = 0; i < nx; ++i)
        for (int k = 0; k < nz; ++k) plan_exec(&py, a + i * sx + k, sy);
    for (int j = 0; j < ny; ++j)
        for (int k = 0; k < nz; ++k) plan_exec(&px, a + j * sy + k, sx);

    plan_free(&pz);
    plan_free(&py);
    plan_free(&px);
    return ODGPE_OK;
}

/* ------------------------------------------------------------------------------------ */
/* handle                                                                                */
/* ------------------------------------------------------------------------------------ */

static double axis_d(const odgpe_handle *h, int a) { return a == 0 ? h->dx : (a == 1 ? h->dy : h->dz); }
static int axis_n(const odgpe_handle *h, int a) { return a == 0 ? h->nx : (a == 1 ? h->ny : h->nz); }

/* grid coordinate (R#6): x_i = (i - n/2) * d */
static double coord(int i, int n, double d) { return (double)(i - n / 2) * d; }

odgpe_handle *odgpe_create(int nx, int ny, int nz, double dx, double dy, double dz, double dt,
                           double gamma, double nu, double lambda, double g, double gdd, int mode)
{
    if (nx < 4 || ny < 4 || nz < 4) return NULL;
    if (!(dx > 0.0) || !(dy > 0.0) || !(dz > 0.0) || !(dt > 0.0)) return NULL;
    if (mode != ODGPE_IMAG && mode != ODGPE_REAL) return NULL;
    odgpe_handle *h = (odgpe_handle *)calloc(1, sizeof(*h));
    if (!h) return NULL;
    h->nx = nx; h->ny = ny; h->nz = nz;
    h->dx = dx; h->dy = dy; h->dz = dz; h->dt = dt;
    h->gamma = gamma; h->nu = nu; h->lambda = lambda;
    h->g = g; h->gdd = gdd; h->mode = mode;

    /* Crank-Nicolson coefficients (R#9):  A psi' = B psi,  A = tridiag(-r, 1+2r, -r),
       B = tridiag(r, 1-2r, r),  r = dt/(4 d^2) (imag)  or  i dt/(4 d^2) (real).
       Thomas elimination factors for the constant-coefficient matrix A on unknowns 1..n-2:
         inv_1 = 1/(1+2r),  c_1 = -r inv_1;  inv_j = 1/((1+2r) + r c_{j-1}),  c_j = -r inv_j. */
    for (int a = 0; a < 3; ++a) {
        int n = axis_n(h, a);
        double d = axis_d(h, a);
        double rr = dt / (4.0 * d * d);
        cplx r = (mode == ODGPE_IMAG) ? (cplx)rr : rr * I;
        h->r[a] = r;
        h->inv[a] = (cplx *)malloc(sizeof(cplx) * (size_t)n);
        h->c[a] = (cplx *)malloc(sizeof(cplx) * (size_t)n);
        if (!h->inv[a] || !h->c[a]) { odgpe_destroy(h); return NULL; }
        for (int j = 0; j < n; ++j) { h->inv[a][j] = 0.0; h->c[a][j] = 0.0; }
        cplx diag = 1.0 + 2.0 * r;
        h->inv[a][1] = 1.0 / diag;
        h->c[a][1] = -r * h->inv[a][1];
        for (int j = 2; j <= n - 2; ++j) {
            h->inv[a][j] = 1.0 / (diag + r * h->c[a][j - 1]);
            h->c[a][j] = -r * h->inv[a][j];
        }
    }
    return h;
}

void odgpe_destroy(odgpe_handle *h)
{
    if (!h) return;
    for (int a = 0; a < 3; ++a) { free(h->inv[a]); free(h->c[a]); }
    free(h);
}

/* ------------------------------------------------------------------------------------ */
/* step 2: dipolar mean field by the convolution theorem                         */
/* ------------------------------------------------------------------------------------ */

/* wave number of DFT bin m (R#10, R#11): k = 2 pi f/(n d), f = m for m <= n/2 else m - n */
static double wavenum(int m, int n, double d)
{
    int f = (m <= n / 2) ? m : m - n;
    return 2.0 * ODGPE_PI * (double)f / ((double)n * d);
}

int odgpe_dipolar(odgpe_handle *h, const double *dens, double *phi)
{
    if (!h || !dens || !phi) return ODGPE_ERR_ARG;
    size_t N = (size_t)h->nx * h->ny * h->nz;
    cplx *a = (cplx *)malloc(sizeof(cplx) * N);
    if (!a) return ODGPE_ERR_NOMEM;
    for (size_t p = 0; p < N; ++p) a[p] = dens[p];
    int rc = odgpe_dft3(h->nx, h->ny, h->nz, a, -1);
    if (rc != ODGPE_OK) { free(a); return rc; }
    for (int i = 0; i < h->nx; ++i) {
        double kx = wavenum(i, h->nx, h->dx);
        for (int j = 0; j < h->ny; ++j) {
            double ky = wavenum(j, h->ny, h->dy);
            for (int k = 0; k < h->nz; ++k) {
                double kz = wavenum(k, h->nz, h->dz);
                double k2 = kx * kx + ky * ky + kz * kz;
                double u = 0.0;                                  /* Udd(0) = 0, BJ:configs[0] */
                if (i != 0 || j != 0 || k != 0)
                    u = (4.0 * ODGPE_PI / 3.0) * (3.0 * kz * kz / k2 - 1.0);
                a[((size_t)i * h->ny + j) * h->nz + k] *= u;
            }
        }
    }
    rc = odgpe_dft3(h->nx, h->ny, h->nz, a, +1);
    if (rc != ODGPE_OK) { free(a); return rc; }
    double invN = 1.0 / (double)N;
    for (size_t p = 0; p < N; ++p) phi[p] = creal(a[p]) * invN;
    free(a);
    return ODGPE_OK;
}

/* ------------------------------------------------------------------------------------ */
/* steps 1-3: density, Phi, nonlinear / potential exponential (BJ:north_star (a),(b))    */
/* ------------------------------------------------------------------------------------ */

int odgpe_nonlinear(odgpe_handle *h, double complex *psi)
{
    if (!h || !psi) return ODGPE_ERR_ARG;
    size_t N = (size_t)h->nx * h->ny * h->nz;
    double *dens = (double *)malloc(sizeof(double) * N);
    double *phi = (double *)malloc(sizeof(double) * N);
    if (!dens || !phi) { free(dens); free(phi); return ODGPE_ERR_NOMEM; }
    for (size_t p = 0; p < N; ++p)
        dens[p] = creal(psi[p]) * creal(psi[p]) + cimag(psi[p]) * cimag(psi[p]);
    int rc = odgpe_dipolar(h, dens, phi);
    if (rc != ODGPE_OK) { free(dens); free(phi); return rc; }
    for (int i = 0; i < h->nx; ++i) {
        double x = coord(i, h->nx, h->dx);
        for (int j = 0; j < h->ny; ++j) {
            double y = coord(j, h->ny, h->dy);
            for (int k = 0; k < h->nz; ++k) {
                double z = coord(k, h->nz, h->dz);
                size_t p = ((size_t)i * h->ny + j) * h->nz + k;
                double V = 0.5 * (h->gamma * h->gamma * x * x + h->nu * h->nu * y * y +
                                  h->lambda * h->lambda * z * z);
                double H = V + h->g * dens[p] + h->gdd * phi[p];
                if (h->mode == ODGPE_IMAG) {
                    psi[p] = exp(-h->dt * H) * psi[p];           /* R#18: no clamp */
                } else {
                    double ph = h->dt * H;
                    psi[p] = (cos(ph) - sin(ph) * I) * psi[p];
                }
            }
        }
    }
    free(dens);
    free(phi);
    return ODGPE_OK;
}

/* ------------------------------------------------------------------------------------ */
/* step 4: Crank-Nicolson line solve (BJ:north_star (c); R#7, R#9)                       */
/*   end nodes are the Dirichlet boundary: treated as 0 on input, written as 0 on output */
/* ------------------------------------------------------------------------------------ */

static void cn_line(const odgpe_handle *h, int axis, cplx *p, size_t stride, cplx *d, cplx *e)
{
    int n = axis_n(h, axis);
    cplx r = h->r[axis];
    const cplx *inv = h->inv[axis];
    const cplx *c = h->c[axis];
    /* right-hand side d = B psi on j = 1..n-2 with psi_0 = psi_{n-1} = 0 */
    for (int j = 1; j <= n - 2; ++j) {
        cplx lo = (j == 1) ? 0.0 : p[(size_t)(j - 1) * stride];
        cplx hi = (j == n - 2) ? 0.0 : p[(size_t)(j + 1) * stride];
        d[j] = r * lo + (1.0 - 2.0 * r) * p[(size_t)j * stride] + r * hi;
    }
    /* forward elimination */
    e[1] = d[1] * inv[1];
    for (int j = 2; j <= n - 2; ++j) e[j] = (d[j] + r * e[j - 1]) * inv[j];
    /* back substitution */
    p[(size_t)(n - 2) * stride] = e[n - 2];
    for (int j = n - 3; j >= 1; --j) p[(size_t)j * stride] = e[j] - c[j] * p[(size_t)(j + 1) * stride];
    p[0] = 0.0;
    p[(size_t)(n - 1) * stride] = 0.0;
}

int odgpe_sweep(odgpe_handle *h, double complex *psi, int axis)
{
    if (!h || !psi || axis < 0 || axis > 2) return ODGPE_ERR_ARG;
    int n = axis_n(h, axis);
    cplx *d = (cplx *)malloc(sizeof(cplx) * (size_t)n);
    cplx *e = (cplx *)malloc(sizeof(cplx) * (size_t)n);
    if (!d || !e) { free(d); free(e); return ODGPE_ERR_NOMEM; }
    size_t sy = (size_t)h->nz, sx = (size_t)h->ny * h->nz;
    if (axis == 0) {
        for (int j = 0; j < h->ny; ++j)
            for (int k = 0; k < h->nz; ++k) cn_line(h, 0, psi + j * sy + k, sx, d, e);
    } else if (axis == 1) {
        for (int i = 0; i < h->nx; ++i)
            for (int k = 0; k < h->nz; ++k) cn_line(h, 1, psi + i * sx + k, sy, d, e);
    } else {
        for (int i = 0; i < h->nx; ++i)
            for (int j = 0; j < h->ny; ++j) cn_line(h, 2, psi + i * sx + j * sy, 1, d, e);
    }
    free(d);
    free(e);
    return ODGPE_OK;
}

/* ------------------------------------------------------------------------------------ */
/* observables (R#14-R#17): plain sums times dV                                           */
/* ------------------------------------------------------------------------------------ */

static double abs2(cplx z) { return creal(z) * creal(z) + cimag(z) * cimag(z); }

int odgpe_norm(odgpe_handle *h, const double complex *psi, double *norm)
{
    if (!h || !psi || !norm) return ODGPE_ERR_ARG;
    size_t N = (size_t)h->nx * h->ny * h->nz;
    double s = 0.0;
    for (size_t p = 0; p < N; ++p) s += abs2(psi[p]);
    *norm = s * h->dx * h->dy * h->dz;
    return ODGPE_OK;
}

int odgpe_rms(odgpe_handle *h, const double complex *psi, double rms[4])
{
    if (!h || !psi || !rms) return ODGPE_ERR_ARG;
    double sx2 = 0.0, sy2 = 0.0, sz2 = 0.0, s = 0.0;
    for (int i = 0; i < h->nx; ++i) {
        double x = coord(i, h->nx, h->dx);
        for (int j = 0; j < h->ny; ++j) {
            double y = coord(j, h->ny, h->dy);
            for (int k = 0; k < h->nz; ++k) {
                double z = coord(k, h->nz, h->dz);
                double n = abs2(psi[((size_t)i * h->ny + j) * h->nz + k]);
                s += n;
                sx2 += x * x * n;
                sy2 += y * y * n;
                sz2 += z * z * n;
            }
        }
    }
    rms[0] = sqrt(sx2 / s);
    rms[1] = sqrt(sy2 / s);
    rms[2] = sqrt(sz2 / s);
    rms[3] = sqrt((sx2 + sy2 + sz2) / s);
    return ODGPE_OK;
}

int odgpe_energy_terms(odgpe_handle *h, const double complex *psi, double out[4])
{
    if (!h || !psi || !out) return ODGPE_ERR_ARG;
    int nx = h->nx, ny = h->ny, nz = h->nz;
    size_t N = (size_t)nx * ny * nz;
    size_t sy = (size_t)nz, sx = (size_t)ny * nz;
    double *dens = (double *)malloc(sizeof(double) * N);
    double *phi = (double *)malloc(sizeof(double) * N);
    if (!dens || !phi) { free(dens); free(phi); return ODGPE_ERR_NOMEM; }
    for (size_t p = 0; p < N; ++p) dens[p] = abs2(psi[p]);
    int rc = odgpe_dipolar(h, dens, phi);
    if (rc != ODGPE_OK) { free(dens); free(phi); return rc; }

    /* kinetic term (R#16): T = sum_a (1/2) sum_links |psi_{j+1} - psi_j|^2 / d_a^2,
       links j = -1..n-1 with psi_{-1} = psi_n = 0 */
    double tx = 0.0, ty = 0.0, tz = 0.0;
    for (int i = 0; i < nx; ++i)
        for (int j = 0; j < ny; ++j)
            for (int k = 0; k < nz; ++k) {
                size_t p = i * sx + j * sy + k;
                cplx here = psi[p];
                cplx px = (i + 1 < nx) ? psi[p + sx] : 0.0;
                cplx py = (j + 1 < ny) ? psi[p + sy] : 0.0;
                cplx pz = (k + 1 < nz) ? psi[p + 1] : 0.0;
                tx += abs2(px - here);
                ty += abs2(py - here);
                tz += abs2(pz - here);
                if (i == 0) tx += abs2(here);                   /* link from the ghost at -1 */
                if (j == 0) ty += abs2(here);
                if (k == 0) tz += abs2(here);
            }
    double T = 0.5 * (tx / (h->dx * h->dx) + ty / (h->dy * h->dy) + tz / (h->dz * h->dz));

    double sV = 0.0, sg = 0.0, sdd = 0.0, s = 0.0;
    for (int i = 0; i < nx; ++i) {
        double x = coord(i, nx, h->dx);
        for (int j = 0; j < ny; ++j) {
            double y = coord(j, ny, h->dy);
            for (int k = 0; k < nz; ++k) {
                double z = coord(k, nz, h->dz);
                size_t p = i * sx + j * sy + k;
                double V = 0.5 * (h->gamma * h->gamma * x * x + h->nu * h->nu * y * y +
                                  h->lambda * h->lambda * z * z);
                double n = dens[p];
                s += n;
                sV += V * n;
                sg += n * n;
                sdd += phi[p] * n;
            }
        }
    }
    /* the dV factors of numerator and norm cancel; the density entering g n and gdd Phi is
       the one given (not renormalised), as in the step itself */
    out[0] = T / s;
    out[1] = sV / s;
    out[2] = h->g * sg / s;
    out[3] = h->gdd * sdd / s;
    free(dens);
    free(phi);
    return ODGPE_OK;
}

int odgpe_chempot(odgpe_handle *h, const double complex *psi, double *mu)
{
    double t[4];
    if (!mu) return ODGPE_ERR_ARG;
    int rc = odgpe_energy_terms(h, psi, t);
    if (rc != ODGPE_OK) return rc;
    *mu = t[0] + t[1] + t[2] + t[3];
    return ODGPE_OK;
}

int odgpe_energy(odgpe_handle *h, const double complex *psi, double *energy)
{
    double t[4];
    if (!energy) return ODGPE_ERR_ARG;
    int rc = odgpe_energy_terms(h, psi, t);
    if (rc != ODGPE_OK) return rc;
    *energy = t[0] + t[1] + 0.5 * t[2] + 0.5 * t[3];
    return ODGPE_OK;
}

/* ------------------------------------------------------------------------------------ */
/* the step (BJ:north_star; R#3: N(dt), K_x(dt), K_y(dt), K_z(dt), renormalise)          */
/* ------------------------------------------------------------------------------------ */

int odgpe_step(odgpe_handle *h, double complex *psi, int nsteps)
{
    if (!h || !psi || nsteps < 0) return ODGPE_ERR_ARG;
    size_t N = (size_t)h->nx * h->ny * h->nz;
    int status = ODGPE_OK;
    for (int s = 0; s < nsteps; ++s) {
        int rc = odgpe_nonlinear(h, psi);
        if (rc != ODGPE_OK) return rc;
        for (int a = 0; a < 3; ++a) {
            rc = odgpe_sweep(h, psi, a);
            if (rc != ODGPE_OK) return rc;
        }
        if (h->mode == ODGPE_IMAG) {
            double norm;
            odgpe_norm(h, psi, &norm);
            if (!(norm > 0.0) || !isfinite(norm)) status = ODGPE_ERR_NONFINITE;
            double sq = sqrt(norm);
            for (size_t p = 0; p < N; ++p) psi[p] = psi[p] / sq;
        }
    }
    return status;
}
