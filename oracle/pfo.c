/*
 * pfo.c -- ORACLE (test infrastructure, not the product). See pfo.h for scope, pins and citations.
 * Plain C99, fp64, libm only; optional OpenMP over independent lines / points (no algorithmic change).
 */
#include "pfo.h"

#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#ifndef M_PI
#define M_PI 3.14159265358979323846264338327950288
#endif

#define PFO_MAX_ETA 64

int pfo_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

static long pfo_npoints(const pfo_params *p) { return (long)p->n[0] * p->n[1] * p->n[2]; }

static int pfo_check(const pfo_params *p)
{
    if (!p) return -1;
    if (p->ndim != 2 && p->ndim != 3) return -1;
    if (p->n[0] < 1 || p->n[1] < 1 || p->n[2] < 1) return -1;
    if (p->ndim == 2 && p->n[2] != 1) return -1;
    if (p->n_eta < 0 || p->n_eta > PFO_MAX_ETA) return -1;
    for (int d = 0; d < p->ndim; ++d) if (!(p->dx[d] > 0.0)) return -1;
    return 0;
}

/* ------------------------------------------------------------------------------------------
 * Pointwise model.
 *   h(eta)  = sum_i eta_i^3 (6 eta_i^2 - 15 eta_i + 10)
 *   g(eta)  = sum_i eta_i^2 (1 - eta_i)^2 + alpha sum_i sum_{j != i} eta_i^2 eta_j^2
 *   f^alpha = rho^2 (c - c_alpha)^2,  f^beta = rho^2 (c_beta - c)^2
 *   f_chem  = f^alpha (1 - h) + f^beta h + w g
 * ---------------------------------------------------------------------------------------- */
double pfo_fchem(const pfo_params *p, double c, const double *eta)
{
    double h = 0.0, g = 0.0;
    for (int i = 0; i < p->n_eta; ++i) {
        double e = eta[i];
        h += e * e * e * (6.0 * e * e - 15.0 * e + 10.0);
        g += e * e * (1.0 - e) * (1.0 - e);
        for (int j = 0; j < p->n_eta; ++j)            /* ordered double sum, exactly as printed */
            if (j != i) g += p->alpha * e * e * eta[j] * eta[j];
    }
    double fa = p->rho2 * (c - p->c_alpha) * (c - p->c_alpha);
    double fb = p->rho2 * (p->c_beta - c) * (p->c_beta - c);
    return fa * (1.0 - h) + fb * h + p->w * g;
}

/* Derivatives of the expressions above (not printed in the paper):
 *   d f/dc      = 2 rho^2 (c - c_alpha)(1 - h) - 2 rho^2 (c_beta - c) h
 *   d h/deta_i  = 30 eta_i^2 (1 - eta_i)^2
 *   d g/deta_i  = 2 eta_i (1 - eta_i)(1 - 2 eta_i) + 4 alpha eta_i sum_{j != i} eta_j^2
 *                 (each unordered pair occurs twice in the ordered double sum -> 4 alpha)
 *   d f/deta_i  = (f^beta - f^alpha) dh/deta_i + w dg/deta_i                                  */
void pfo_dfchem(const pfo_params *p, double c, const double *eta, double *dfdc, double *dfdeta)
{
    double h = 0.0, s2 = 0.0;
    for (int i = 0; i < p->n_eta; ++i) {
        double e = eta[i];
        h  += e * e * e * (6.0 * e * e - 15.0 * e + 10.0);
        s2 += e * e;
    }
    double fa = p->rho2 * (c - p->c_alpha) * (c - p->c_alpha);
    double fb = p->rho2 * (p->c_beta - c) * (p->c_beta - c);
    *dfdc = 2.0 * p->rho2 * (c - p->c_alpha) * (1.0 - h) - 2.0 * p->rho2 * (p->c_beta - c) * h;
    for (int i = 0; i < p->n_eta; ++i) {
        double e  = eta[i];
        double dh = 30.0 * e * e * (1.0 - e) * (1.0 - e);
        double dg = 2.0 * e * (1.0 - e) * (1.0 - 2.0 * e) + 4.0 * p->alpha * e * (s2 - e * e);
        dfdeta[i] = (fb - fa) * dh + p->w * dg;
    }
}

/* ------------------------------------------------------------------------------------------
 * Discrete Fourier transforms. Forward sign e^{-i xi x} (Eq. 9 convention:
 * grad f -> i xi f^ corresponds to f(x) = sum f^ e^{+i xi x}).
 * ---------------------------------------------------------------------------------------- */
void pfo_dft1d_naive(int n, const double *in, double *out, int sign)
{
    for (int k = 0; k < n; ++k) {
        double sr = 0.0, si = 0.0;
        for (int j = 0; j < n; ++j) {
            /* reduce jk mod n in integers so the angle stays accurate for large n */
            long   m  = ((long)j * (long)k) % (long)n;
            double a  = (double)sign * 2.0 * M_PI * (double)m / (double)n;
            double wr = cos(a), wi = sin(a);
            sr += in[2 * j] * wr - in[2 * j + 1] * wi;
            si += in[2 * j] * wi + in[2 * j + 1] * wr;
        }
        out[2 * k] = sr; out[2 * k + 1] = si;
    }
}

/* Textbook iterative radix-2 decimation-in-time Cooley-Tukey: bit-reversal permutation followed
 * by log2(n) butterfly stages; every twiddle is evaluated directly with cos/sin. */
void pfo_fft1d_radix2(int n, double *data, int sign)
{
    for (int i = 1, j = 0; i < n; ++i) {
        int bit = n >> 1;
        for (; j & bit; bit >>= 1) j ^= bit;
        j ^= bit;
        if (i < j) {
            double tr = data[2 * i], ti = data[2 * i + 1];
            data[2 * i] = data[2 * j]; data[2 * i + 1] = data[2 * j + 1];
            data[2 * j] = tr;          data[2 * j + 1] = ti;
        }
    }
    for (int len = 2; len <= n; len <<= 1) {
        int half = len >> 1;
        for (int start = 0; start < n; start += len) {
            for (int k = 0; k < half; ++k) {
                double a  = (double)sign * 2.0 * M_PI * (double)k / (double)len;
                double wr = cos(a), wi = sin(a);
                double *u = data + 2 * (start + k);
                double *v = data + 2 * (start + k + half);
                double tr = v[0] * wr - v[1] * wi;
                double ti = v[0] * wi + v[1] * wr;
                v[0] = u[0] - tr; v[1] = u[1] - ti;
                u[0] = u[0] + tr; u[1] = u[1] + ti;
            }
        }
    }
}

static int pfo_is_pow2(int n) { return n >= 1 && (n & (n - 1)) == 0; }

/* Row-column transform: for each axis, every line along that axis is copied out, transformed
 * and copied back. data is interleaved complex, index ((z*ny + y)*nx + x). */
int pfo_fftn(const int n[3], double *data, int sign, int naive)
{
    const long nx = n[0], ny = n[1], nz = n[2];
    const long stride[3] = { 1, nx, nx * ny };
    for (int axis = 0; axis < 3; ++axis) {
        const int len = n[axis];
        if (len == 1) continue;
        if (!naive && !pfo_is_pow2(len)) return -1;
        const long nlines = nx * ny * nz / len;
        int fail = 0;
#ifdef _OPENMP
#pragma omp parallel
#endif
        {
            double *line = (double *)malloc(sizeof(double) * 2 * (size_t)len);
            double *tmp  = (double *)malloc(sizeof(double) * 2 * (size_t)len);
            if (!line || !tmp) {
#ifdef _OPENMP
#pragma omp atomic write
#endif
                fail = 1;
            } else {
#ifdef _OPENMP
#pragma omp for schedule(static)
#endif
                for (long l = 0; l < nlines; ++l) {
                    /* base index of line l: enumerate the two other axes */
                    long base;
                    if (axis == 0)      base = l * nx;                                  /* l = z*ny + y */
                    else if (axis == 1) base = (l / nx) * nx * ny + (l % nx);           /* l = z*nx + x */
                    else                base = l;                                       /* l = y*nx + x */
                    for (int j = 0; j < len; ++j) {
                        line[2 * j]     = data[2 * (base + j * stride[axis])];
                        line[2 * j + 1] = data[2 * (base + j * stride[axis]) + 1];
                    }
                    if (naive) { pfo_dft1d_naive(len, line, tmp, sign); memcpy(line, tmp, sizeof(double) * 2 * (size_t)len); }
                    else       { pfo_fft1d_radix2(len, line, sign); }
                    for (int j = 0; j < len; ++j) {
                        data[2 * (base + j * stride[axis])]     = line[2 * j];
                        data[2 * (base + j * stride[axis]) + 1] = line[2 * j + 1];
                    }
                }
            }
            free(line); free(tmp);
        }
        if (fail) return -1;
    }
    return 0;
}

/* ------------------------------------------------------------------------------------------
 * Frequencies. Index vector [0, ..., n/2, -(n/2-1), ..., -1], l = n dx,
 * xi = 2 pi m / l.
 * ---------------------------------------------------------------------------------------- */
double pfo_k2_axis(int kind, int n, double dx, int idx)
{
    int    m  = (idx <= n / 2) ? idx : idx - n;
    double l  = (double)n * dx;
    double xi = 2.0 * M_PI * (double)m / l;
    if (kind == 0) return xi * xi;                                                       /* Eq. 16/19 */
    if (kind == 1) return -2.0 * (cos(dx * xi) - 1.0) / (dx * dx);                       /* Eq. 17/20 */
    return -(16.0 * cos(dx * xi) - cos(2.0 * dx * xi) - 15.0) / (6.0 * dx * dx);         /* Eq. 18/21 */
}

/* 5-/7-point Laplacian with periodic wrap (second-order centred, regular grid). */
void pfo_laplacian(const pfo_params *p, const double *u, double *out)
{
    const long nx = p->n[0], ny = p->n[1], nz = p->n[2];
    const double ax = 1.0 / (p->dx[0] * p->dx[0]);
    const double ay = 1.0 / (p->dx[1] * p->dx[1]);
    const double az = (p->ndim == 3) ? 1.0 / (p->dx[2] * p->dx[2]) : 0.0;
#ifdef _OPENMP
#pragma omp parallel for collapse(2) schedule(static)
#endif
    for (long z = 0; z < nz; ++z)
        for (long y = 0; y < ny; ++y)
            for (long x = 0; x < nx; ++x) {
                long xm = (x + nx - 1) % nx, xp = (x + 1) % nx;
                long ym = (y + ny - 1) % ny, yp = (y + 1) % ny;
                long i  = (z * ny + y) * nx + x;
                double v = u[i];
                double s = ax * (u[(z * ny + y) * nx + xp] + u[(z * ny + y) * nx + xm] - 2.0 * v)
                         + ay * (u[(z * ny + yp) * nx + x] + u[(z * ny + ym) * nx + x] - 2.0 * v);
                if (p->ndim == 3) {
                    long zm = (z + nz - 1) % nz, zp = (z + 1) % nz;
                    s += az * (u[(zp * ny + y) * nx + x] + u[(zm * ny + y) * nx + x] - 2.0 * v);
                }
                out[i] = s;
            }
}

/* g = d f_chem/dc and h_i = d f_chem/d eta_i at every grid point (Alg. 1). */
static void pfo_eval_derivatives(const pfo_params *p, const double *c, const double *eta, double *g, double *h)
{
    const long N = pfo_npoints(p);
#ifdef _OPENMP
#pragma omp parallel for schedule(static)
#endif
    for (long i = 0; i < N; ++i) {
        double e[PFO_MAX_ETA], de[PFO_MAX_ETA], dc;
        for (int k = 0; k < p->n_eta; ++k) e[k] = eta[(long)k * N + i];
        pfo_dfchem(p, c[i], e, &dc, de);
        g[i] = dc;
        for (int k = 0; k < p->n_eta; ++k) h[(long)k * N + i] = de[k];
    }
}

static void pfo_real_to_complex(long N, const double *re, double *z)
{
    for (long i = 0; i < N; ++i) { z[2 * i] = re[i]; z[2 * i + 1] = 0.0; }
}

/* ------------------------------------------------------------------------------------------
 * Semi-implicit Fourier-spectral step, Algorithm 1:
 *   g^ = F[df/dc], h_i^ = F[df/deta_i]
 *   b_c^   = c^  - M dt |xi|^2 g^          (Eq. 12)
 *   b_eta^ = eta^ - L dt h_i^              (Eq. 13)
 *   c^   <- b_c^   / (1 + M dt kappa_c |xi|^4)      (Eq. 14; Alg. 1 prints |xi|^2
 *                                                   there -- a typo, Eq. 10/14 have |xi|^4)
 *   eta^ <- b_eta^ / (1 + L dt kappa_eta |xi|^2)    (Eq. 15)
 *   c, eta_i = F^-1[...]
 * The real fields are re-transformed each step (the paper carries c^; same result to rounding).
 * ---------------------------------------------------------------------------------------- */
int pfo_step_fs(const pfo_params *p, double *c, double *eta, int nsteps)
{
    if (pfo_check(p) || !c || (p->n_eta > 0 && !eta) || nsteps < 0) return -1;
    const long N = pfo_npoints(p);
    const long nx = p->n[0], ny = p->n[1], nz = p->n[2];
    const int  F = 1 + p->n_eta;
    double *g   = (double *)malloc(sizeof(double) * (size_t)N * (size_t)F);      /* g, h_1..h_p */
    double *uh  = (double *)malloc(sizeof(double) * 2 * (size_t)N);
    double *gh  = (double *)malloc(sizeof(double) * 2 * (size_t)N);
    double *k2x = (double *)malloc(sizeof(double) * (size_t)nx);
    double *k2y = (double *)malloc(sizeof(double) * (size_t)ny);
    double *k2z = (double *)malloc(sizeof(double) * (size_t)nz);
    int rc = 0;
    if (!g || !uh || !gh || !k2x || !k2y || !k2z) { rc = -1; goto done; }

    /* |xi|^2 is computed once, before the time loop. */
    for (long i = 0; i < nx; ++i) k2x[i] = pfo_k2_axis(p->k2_kind, (int)nx, p->dx[0], (int)i);
    for (long i = 0; i < ny; ++i) k2y[i] = pfo_k2_axis(p->k2_kind, (int)ny, p->dx[1], (int)i);
    for (long i = 0; i < nz; ++i) k2z[i] = (p->ndim == 3) ? pfo_k2_axis(p->k2_kind, (int)nz, p->dx[2], (int)i) : 0.0;

    for (int step = 0; step < nsteps; ++step) {
        pfo_eval_derivatives(p, c, eta, g, g + N);
        for (int f = 0; f < F; ++f) {
            double *u = (f == 0) ? c : eta + (long)(f - 1) * N;
            pfo_real_to_complex(N, u, uh);
            pfo_real_to_complex(N, g + (long)f * N, gh);
            if (pfo_fftn(p->n, uh, -1, p->dft_kind) || pfo_fftn(p->n, gh, -1, p->dft_kind)) { rc = -1; goto done; }
#ifdef _OPENMP
#pragma omp parallel for collapse(2) schedule(static)
#endif
            for (long z = 0; z < nz; ++z)
                for (long y = 0; y < ny; ++y)
                    for (long x = 0; x < nx; ++x) {
                        long   i  = (z * ny + y) * nx + x;
                        double k2 = k2x[x] + k2y[y] + k2z[z];
                        if (f == 0) {
                            double k4  = k2 * k2;
                            double den = 1.0 + p->M * p->dt * p->kappa_c * k4;
                            double br  = uh[2 * i]     - p->M * p->dt * k2 * gh[2 * i];
                            double bi  = uh[2 * i + 1] - p->M * p->dt * k2 * gh[2 * i + 1];
                            uh[2 * i] = br / den; uh[2 * i + 1] = bi / den;
                        } else {
                            double den = 1.0 + p->L * p->dt * p->kappa_eta * k2;
                            double br  = uh[2 * i]     - p->L * p->dt * gh[2 * i];
                            double bi  = uh[2 * i + 1] - p->L * p->dt * gh[2 * i + 1];
                            uh[2 * i] = br / den; uh[2 * i + 1] = bi / den;
                        }
                    }
            if (pfo_fftn(p->n, uh, +1, p->dft_kind)) { rc = -1; goto done; }
            for (long i = 0; i < N; ++i) u[i] = uh[2 * i] / (double)N;          /* real part, 1/N on the inverse */
        }
    }
done:
    free(g); free(uh); free(gh); free(k2x); free(k2y); free(k2z);
    return rc;
}

/* ------------------------------------------------------------------------------------------
 * Explicit FD step: three "kernels", all right-hand sides at time t,
 *   (i)   mu    = df/dc - kappa_c lap c
 *   (ii)  c'    = c + dt M lap mu           (M constant: div(M grad mu) = M lap mu, Eq. 2)
 *   (iii) eta_i'= eta_i - dt L (df/deta_i - kappa_eta lap eta_i)        (Eq. 3)
 * then the "pointer swap" (here: copy back).
 * ---------------------------------------------------------------------------------------- */
int pfo_step_fd(const pfo_params *p, double *c, double *eta, int nsteps)
{
    if (pfo_check(p) || !c || (p->n_eta > 0 && !eta) || nsteps < 0) return -1;
    const long N = pfo_npoints(p);
    const int  F = 1 + p->n_eta;
    double *g   = (double *)malloc(sizeof(double) * (size_t)N * (size_t)F);
    double *mu  = (double *)malloc(sizeof(double) * (size_t)N);
    double *lap = (double *)malloc(sizeof(double) * (size_t)N);
    double *cn  = (double *)malloc(sizeof(double) * (size_t)N);
    if (!g || !mu || !lap || !cn) { free(g); free(mu); free(lap); free(cn); return -1; }
    for (int step = 0; step < nsteps; ++step) {
        pfo_eval_derivatives(p, c, eta, g, g + N);
        pfo_laplacian(p, c, lap);
        for (long i = 0; i < N; ++i) mu[i] = g[i] - p->kappa_c * lap[i];
        pfo_laplacian(p, mu, lap);
        for (long i = 0; i < N; ++i) cn[i] = c[i] + p->dt * p->M * lap[i];
        for (int k = 0; k < p->n_eta; ++k) {
            double *e = eta + (long)k * N;
            const double *hk = g + (long)(k + 1) * N;
            pfo_laplacian(p, e, lap);
            /* e is only read at point i after lap has been fully formed, so in-place is time-t exact */
            for (long i = 0; i < N; ++i) e[i] = e[i] - p->dt * p->L * (hk[i] - p->kappa_eta * lap[i]);
        }
        memcpy(c, cn, sizeof(double) * (size_t)N);
    }
    free(g); free(mu); free(lap); free(cn);
    return 0;
}

/* ------------------------------------------------------------------------------------------
 * Total free energy, Eq. 1, as a Riemann sum with cell volume dV = prod dx.
 * The paper does not say how |grad .|^2 is discretised -> two kinds.
 * ---------------------------------------------------------------------------------------- */
static int pfo_grad_energy(const pfo_params *p, const double *u, int kind, double *out)
{
    const long nx = p->n[0], ny = p->n[1], nz = p->n[2];
    const long N = nx * ny * nz;
    double dV = p->dx[0] * p->dx[1] * (p->ndim == 3 ? p->dx[2] : 1.0);
    double s = 0.0;
    if (kind == 1) {
        for (long z = 0; z < nz; ++z)
            for (long y = 0; y < ny; ++y)
                for (long x = 0; x < nx; ++x) {
                    long i = (z * ny + y) * nx + x;
                    double dxu = (u[(z * ny + y) * nx + (x + 1) % nx] - u[i]) / p->dx[0];
                    double dyu = (u[(z * ny + (y + 1) % ny) * nx + x] - u[i]) / p->dx[1];
                    double dzu = (p->ndim == 3) ? (u[(((z + 1) % nz) * ny + y) * nx + x] - u[i]) / p->dx[2] : 0.0;
                    s += dxu * dxu + dyu * dyu + dzu * dzu;
                }
        *out = s * dV;
        return 0;
    }
    /* Parseval: sum_x |grad u|^2 = (1/N) sum_k |xi|^2 |u^_k|^2 */
    double *uh = (double *)malloc(sizeof(double) * 2 * (size_t)N);
    if (!uh) return -1;
    pfo_real_to_complex(N, u, uh);
    if (pfo_fftn(p->n, uh, -1, p->dft_kind)) { free(uh); return -1; }
    for (long z = 0; z < nz; ++z)
        for (long y = 0; y < ny; ++y)
            for (long x = 0; x < nx; ++x) {
                long i = (z * ny + y) * nx + x;
                double k2 = pfo_k2_axis(p->k2_kind, (int)nx, p->dx[0], (int)x)
                          + pfo_k2_axis(p->k2_kind, (int)ny, p->dx[1], (int)y)
                          + (p->ndim == 3 ? pfo_k2_axis(p->k2_kind, (int)nz, p->dx[2], (int)z) : 0.0);
                s += k2 * (uh[2 * i] * uh[2 * i] + uh[2 * i + 1] * uh[2 * i + 1]);
            }
    free(uh);
    *out = s / (double)N * dV;
    return 0;
}

int pfo_free_energy(const pfo_params *p, const double *c, const double *eta, int gradient_kind, double *out)
{
    if (pfo_check(p) || !c || (p->n_eta > 0 && !eta) || !out) return -1;
    if (gradient_kind != 0 && gradient_kind != 1) return -1;
    const long N = pfo_npoints(p);
    double dV = p->dx[0] * p->dx[1] * (p->ndim == 3 ? p->dx[2] : 1.0);
    double chem = 0.0;
    for (long i = 0; i < N; ++i) {
        double e[PFO_MAX_ETA];
        for (int k = 0; k < p->n_eta; ++k) e[k] = eta[(long)k * N + i];
        chem += pfo_fchem(p, c[i], e);
    }
    out[1] = chem * dV;
    double ge;
    if (pfo_grad_energy(p, c, gradient_kind, &ge)) return -1;
    out[2] = 0.5 * p->kappa_c * ge;
    double total = out[1] + out[2];
    for (int k = 0; k < p->n_eta; ++k) {
        if (pfo_grad_energy(p, eta + (long)k * N, gradient_kind, &ge)) return -1;
        out[3 + k] = 0.5 * p->kappa_eta * ge;
        total += out[3 + k];
    }
    out[0] = total;
    return 0;
}

/* ------------------------------------------------------------------------------------------
 * Eq. 22: E_phi = int (phi_0 - phi)^2 dV / int phi_0^2 dV on a uniform grid.
 * ---------------------------------------------------------------------------------------- */
double pfo_error_eq22(long n, const double *phi, const double *ref)
{
    if (n <= 0 || !phi || !ref) return -1.0;
    double num = 0.0, den = 0.0;
    for (long i = 0; i < n; ++i) {
        double d = ref[i] - phi[i];
        num += d * d;
        den += ref[i] * ref[i];
    }
    if (!(den > 0.0)) return -1.0;
    return num / den;
}
