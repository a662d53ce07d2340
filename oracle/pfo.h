/*
 * pfo.h -- ORACLE (test infrastructure, not the product).
 *
 * A plain, slow, fp64, CPU implementation of the method of
 *   Boccardo, Tong, Leen, Tourret, Segurado, "Efficiency and accuracy of GPU-parallelized
 *   Fourier spectral methods for solving phase-field models" (arXiv 2306.04322),
 * written from the paper's text only (PAPER.md line numbers are cited at every function).
 *
 * It shares NO code with the CUDA path under paper_2306_04322_b200/ and is used only by
 * tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs.
 * There is no blocking, fusion or reordering beyond what the paper states: the semi-implicit
 * step is Algorithm 1 line by line, the transforms are a direct O(n^2) DFT or a textbook
 * radix-2 Cooley-Tukey FFT applied axis by axis on full complex arrays, the FD step is three
 * plain loops.
 *
 * Pins (tests/test_oracle_*.py, all "-m 'not gpu'"): brute-force DFT vs radix-2 vs numpy.fft;
 * central differences of f_chem; closed-form amplification factors of single Fourier modes
 * (FS and FD); conservation of mean c; monotone free energy; 5/7-point Laplacian == F^-1[-|xi_c2|^2 F u];
 * spectral Laplacian exact on band-limited fields; closed-form free-energy integrals (2D and 3D,
 * both gradient kinds); Eq. 22 on cosines of known amplitude; the paper's printed FD time steps
 * against the linear stability bound.
 * Parity unpinned: full trajectories against the paper's figures (Figs. 1-6 are images and the
 * paper's pre-evolved initial fields are not available) -- see DESIGN.md.
 *
 * Layout: every field is a C-contiguous double array [nz][ny][nx], x fastest; eta is
 * [n_eta][nz][ny][nx]. All pointers are host pointers owned by the caller.
 */
#ifndef PFO_H
#define PFO_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct {
    int    ndim;                 /* 2 or 3 */
    int    n[3];                 /* nx, ny, nz (nz = 1 in 2D); any size for the naive DFT, power of two for radix-2 */
    int    n_eta;                /* p: number of Allen-Cahn order parameters (p = 4 in the paper) */
    double dx[3];                /* grid spacing per axis; l_d = n_d * dx_d */
    double dt;                   /* time step */
    double M, L;                 /* mobility and kinetic coefficient, Eqs. 2-3 */
    double kappa_c, kappa_eta;   /* gradient energy coefficients, Eq. 1 */
    double rho2, c_alpha, c_beta, w, alpha;   /* f_chem parameters */
    int    k2_kind;              /* 0: Eq. 16/19 spectral; 1: Eq. 17/20 O(dl^2); 2: Eq. 18/21 O(dl^4) */
    int    dft_kind;             /* 0: radix-2 FFT per axis; 1: direct O(n^2) DFT per axis */
} pfo_params;

/* f_chem = f^alpha (1-h) + f^beta h + w g */
double pfo_fchem(const pfo_params *p, double c, const double *eta);
/* d f_chem / dc and d f_chem / d eta_i, derived from the definitions at PAPER.md:46
 * (the paper does not print them; reading listed in DESIGN.md): dfdeta has n_eta entries. */
void   pfo_dfchem(const pfo_params *p, double c, const double *eta, double *dfdc, double *dfdeta);

/* 1-D transforms on interleaved complex data (re,im,re,im,...).
 * sign = -1: forward, X[k] = sum_j x[j] exp(-2 pi i jk/n); sign = +1: the same with +, UNNORMALISED. */
void   pfo_dft1d_naive (int n, const double *in, double *out, int sign);
void   pfo_fft1d_radix2(int n, double *data, int sign);       /* in place; n must be a power of two */
/* d-dimensional transform of an interleaved complex array [nz][ny][nx], one axis after the other.
 * naive != 0 selects the O(n^2) DFT. The inverse (sign=+1) is UNNORMALISED here. Returns 0 / -1. */
int    pfo_fftn(const int n[3], double *data, int sign, int naive);

/* squared frequency contribution of ONE axis at integer index idx in [0,n):
 * kind 0: (2 pi m / l)^2, m = idx for idx <= n/2 else idx - n         (Eq. 16/19)
 * kind 1: -2 (cos(dx xi) - 1)/dx^2                                   (Eq. 17/20)
 * kind 2: -(16 cos(dx xi) - cos(2 dx xi) - 15)/(6 dx^2)              (Eq. 18/21) */
double pfo_k2_axis(int kind, int n, double dx, int idx);

/* 5-point (2D) / 7-point (3D) periodic Laplacian, second-order centred. */
void   pfo_laplacian(const pfo_params *p, const double *u, double *out);

/* nsteps semi-implicit Fourier-spectral steps, Algorithm 1 with Eqs. 12-15
 * (PAPER.md:103-116); c and eta are updated in place. Returns 0, or -1 on bad arguments. */
int    pfo_step_fs(const pfo_params *p, double *c, double *eta, int nsteps);
/* nsteps explicit forward-Euler finite-difference steps. */
int    pfo_step_fd(const pfo_params *p, double *c, double *eta, int nsteps);

/* Eq. 1 summed over the grid times the cell volume.
 * out[0] total, out[1] chemical, out[2] kappa_c/2 |grad c|^2, out[3+i] kappa_eta/2 |grad eta_i|^2.
 * gradient_kind 0: Parseval with the k2_kind frequencies; 1: forward differences. */
int    pfo_free_energy(const pfo_params *p, const double *c, const double *eta, int gradient_kind, double *out);

/* L2 normalised global error of a field against a reference sampled at the same n points, Eq. 22:
 *   E_phi = int (phi_0 - phi)^2 dV / int phi_0^2 dV = sum (ref - phi)^2 / sum ref^2   (uniform cells: dV cancels).
 * A ratio of squares (no square root), not in percent; the paper's "phase field" is eta = sum_i eta_i.
 * Returns -1.0 on bad arguments or a zero reference. */
double pfo_error_eq22(long n, const double *phi, const double *ref);

/* number of OpenMP threads the loops above will use (1 when built without -fopenmp). */
int    pfo_num_threads(void);

#ifdef __cplusplus
}
#endif
#endif
