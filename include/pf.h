/*
 * pf.h -- C ABI of libpf: the B200 (sm_100a) phase-field stepper.
 *
 * The library advances the coupled Cahn-Hilliard (conserved c) + Allen-Cahn (eta_1..eta_p) model of
 * arXiv 2306.04322 (Boccardo, Tong, Leen, Tourret, Segurado) on a periodic 2D/3D grid:
 *
 *   free energy          F = int f_chem + kappa_c/2 |grad c|^2 + sum_i kappa_eta/2 |grad eta_i|^2   Eq. 1
 *   f_chem               f^alpha (1-h) + f^beta h + w g
 *   Cahn-Hilliard        dc/dt     = div( M grad( df/dc - kappa_c lap c ) )                         Eq. 2
 *   Allen-Cahn           deta_i/dt = -L ( df/deta_i - kappa_eta lap eta_i )                         Eq. 3
 *
 * with either the semi-implicit Fourier-spectral step (Eqs. 12-15; Algorithm 1,
 * PAPER.md:159-193) or the explicit forward-Euler 5/7-point finite-difference step.
 * Every step of both paths runs in hand-written CUDA kernels; there is no CPU fallback: when no
 * CUDA device is usable pf_create returns PF_ECUDA.
 *
 * Conventions
 *   - fields are C-contiguous [nz][ny][nx], x fastest, index (z*ny + y)*nx + x; eta is
 *     [n_eta][nz][ny][nx]; the element type is float (PF_F32) or double (PF_F64) as given in
 *     pf_params.precision; host and device buffers have the same layout;
 *   - `where` says what kind of pointer the caller passes: PF_HOST (pageable or pinned host memory)
 *     or PF_DEVICE (device memory of the context's device). The caller owns its buffers; the library
 *     copies and never keeps a caller pointer after the call returns;
 *   - all work is queued on pf_params.stream (a cudaStream_t passed as void*; borrowed, never destroyed;
 *     NULL = a private blocking stream of the context, which orders with the legacy default stream). pf_step_* and device-side set/get are asynchronous;
 *     pf_get_fields(PF_HOST), pf_set_fields(PF_HOST) and pf_free_energy synchronise that stream;
 *   - a context belongs to the CUDA device that was current in pf_create; every later call must be made with that
 *     device current (PF_EINVAL otherwise);
 *   - every call returns PF_OK (0) or a negative code; nothing throws or aborts. After PF_ECUDA
 *     pf_last_cuda_error gives the CUDA error string.
 */
#ifndef PF_H
#define PF_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct pf_ctx pf_ctx;     /* opaque; owns every device buffer, table and CUDA graph */

enum { PF_F32 = 0, PF_F64 = 1 };
enum { PF_HOST = 0, PF_DEVICE = 1 };
enum { PF_OK = 0, PF_EINVAL = -1, PF_ENOMEM = -2, PF_ECUDA = -3, PF_ESTATE = -4, PF_EUNSUPPORTED = -5 };

typedef struct {
    int    ndim;            /* 2 or 3                                                                         */
    int    n[3];            /* nx (fastest), ny, nz (= 1 when ndim == 2); powers of two, 16 .. 2048            */
    int    n_eta;           /* p, number of Allen-Cahn order parameters, 0 .. 8 (paper: 4)        */
    double dx[3];           /* grid spacing per axis; domain length l_d = n_d * dx_d            */
    double dt;              /* time step                                                                       */
    double M, L;            /* mobility, kinetic coefficient (Eqs. 2-3; paper: 5, 5)                           */
    double kappa_c, kappa_eta;                 /* gradient-energy coefficients (Eq. 1; paper: 3, 3)            */
    double rho2, c_alpha, c_beta, w, alpha;    /* f_chem parameters (paper: 2, .3, .7, 1, 5)   */
    int    precision;       /* PF_F32 | PF_F64: storage and arithmetic type of every kernel                    */
    int    k2_kind;         /* squared frequencies used by the spectral step:
                               0 = Eq. 16/19 (Fourier spectral), 1 = Eq. 17/20 (FS-FD O(dl^2)),
                               2 = Eq. 18/21 (FS-FD O(dl^4))                   */
    void  *stream;          /* cudaStream_t the context runs on (NULL = private blocking stream); borrowed     */
} pf_params;

/* Creates a context on the CURRENT CUDA device: validates p, allocates all device buffers, builds
 * the twiddle and frequency tables. *out is set only on PF_OK.
 * PF_EINVAL: null pointers, ndim not 2/3, dt <= 0, dx <= 0, n_eta out of range, bad enum values;
 * PF_EUNSUPPORTED: a grid size that is not a power of two in 16..2048 (nz must be 1 in 2D); every combination of
 *   grid size, n_eta 0..8 and precision that passes this check can be stepped (tests sweep them);
 * PF_ENOMEM: device allocation failed; PF_ECUDA: no usable device / a CUDA call failed. */
int pf_create(const pf_params *p, pf_ctx **out);

/* Batched small grids (the paper reports that small grids leave the GPU idle: PAPER.md:265, 128^2 "less than 3.8 grid
 * points per CUDA core", 16^3 and 32^3). Creates ONE context that advances nbatch independent replicas of
 * the 2D or 3D problem described by p -- same grid, coefficients and dt, different fields -- with the same kernels and the
 * same number of launches per Fourier-spectral step as a single simulation: the replicas are further rows of the x kernel,
 * further planes of the 3D y kernels and further column blocks of the last-axis kernel. Field arrays of such a context are
 * replica-major:
 *     c: [nbatch][nz][ny][nx],   eta: [nbatch][n_eta][nz][ny][nx]
 * and every replica evolves exactly as it would in its own context (tests compare each with the oracle).
 * pf_step_fs, pf_step_fd, pf_set_fields, pf_get_fields and pf_set_dt work as for a single simulation (pf_step_fd of a 3D
 * batch issues one launch per replica and step); pf_free_energy returns PF_EUNSUPPORTED (read the fields out instead).
 * PF_EINVAL: nbatch outside 1..4096 (and everything pf_create rejects); PF_EUNSUPPORTED: ndim == 3 with nz * nbatch > 65535.
 * nbatch == 1 is pf_create. */
int pf_create_batch(const pf_params *p, int nbatch, pf_ctx **out);

/* Number of replicas of the context (1 for pf_create); 0 for a null pointer. */
int pf_batch_size(const pf_ctx *ctx);

/* Copies the fields into the context (c: [nz][ny][nx]; eta: [n_eta][nz][ny][nx], may be NULL iff
 * n_eta == 0). Invalidates the cached spectral state. */
int pf_set_fields(pf_ctx *ctx, const void *c, const void *eta, int where);

/* nsteps semi-implicit Fourier-spectral steps (Algorithm 1):
 *   g = df_chem/dc, h_i = df_chem/deta_i in real space
 *   c^   <- ( c^   - dt M |xi|^2 g^   ) / ( 1 + dt M kappa_c |xi|^4 )            (Eqs. 12, 14)
 *   eta^ <- ( eta^ - dt L h_i^        ) / ( 1 + dt L kappa_eta |xi|^2 )          (Eqs. 13, 15)
 * with |xi|^2 of k2_kind. The fields are kept in a partially transformed form between steps; the
 * real fields are materialised by pf_get_fields / pf_step_fd / pf_free_energy.
 * Launches: 2 (2D) or 4 (3D) kernels per step, replayed as a CUDA graph of 8 steps for calls of at least 8 steps; square 2D
 * grids up to 64 x 64 run ALL steps of a call of two or more steps in ONE launch (state resident in the shared memory of a
 * thread-block cluster), so one call of n steps is much cheaper there than n calls of one step.
 * nsteps == 0 is a no-op; nsteps < 0 -> PF_EINVAL; no fields set -> PF_ESTATE.
 * Non-finite values are not an error (they propagate). */
int pf_step_fs(pf_ctx *ctx, int nsteps);

/* nsteps explicit forward-Euler steps with the 5-point (2D) / 7-point (3D) Laplacian and periodic
 * wrap-around: mu = df/dc - kappa_c lap c; c += dt M lap mu;
 * eta_i -= dt L (df/deta_i - kappa_eta lap eta_i); every right-hand side at time t. */
int pf_step_fd(pf_ctx *ctx, int nsteps);

/* Copies the current fields out (same layouts as pf_set_fields). With PF_HOST the call returns after
 * the data has arrived. */
int pf_get_fields(pf_ctx *ctx, void *c, void *eta, int where);

/* Eq. 1 as a Riemann sum with cell volume prod(dx), accumulated in fp64.
 * out (HOST pointer, 3 + n_eta doubles): total, chemical, kappa_c/2 |grad c|^2, kappa_eta/2 |grad eta_i|^2 ...
 * gradient_kind 0: spectral, sum_k |xi|^2 |u^_k|^2 / N (Parseval) with the k2_kind frequencies;
 * gradient_kind 1: forward differences (the discretisation the 5/7-point Laplacian derives from). */
int pf_free_energy(pf_ctx *ctx, int gradient_kind, double *out);

/* Free energy for callers that must not allocate device memory.
 *
 * pf_free_energy needs a context, and pf_create pays for a context with a dozen cudaMalloc calls. That rules it out for
 * code that runs where allocating is not an option: a plug-in inside an application whose own memory pool already owns
 * (almost) all of the device, so that a further cudaMalloc fails or takes memory the plug-in has no claim to; an in-situ
 * energy monitor called from another solver's time loop, where cudaMalloc/cudaFree would stall the device on every call;
 * any program with a "nothing is allocated after start-up" rule. pf_free_energy_static serves those callers: no
 * context, no cudaMalloc/cudaFree or other allocating call, ever. Its working memory (per-tile partial sums, a ticket,
 * the result) is a fixed array compiled into libpf.so -- PF_STATIC_SCRATCH_BYTES of global memory that every GPU which
 * loads the library holds until the process exits. The price is a size limit and one shared array.
 *
 * Computes Eq. 1 exactly as pf_free_energy(ctx, gradient_kind = 1, out) does -- f_chem of PAPER.md:46,
 * forward-difference gradients with periodic wrap-around, Riemann sum with cell volume prod(dx), fp64 accumulation --
 * for fields the caller already has on the device.
 *   p    read: ndim, n, n_eta, dx, kappa_c, kappa_eta, rho2, c_alpha, c_beta, w, alpha, precision, stream; the rest
 *        (dt, M, L, k2_kind) is ignored. stream NULL = the legacy default stream;
 *   c    DEVICE pointer (current device), [nz][ny][nx] of float/double per p->precision; read only, caller keeps it;
 *   eta  DEVICE pointer, [n_eta][nz][ny][nx]; may be NULL iff n_eta == 0;
 *   out  HOST pointer, 3 + n_eta doubles: total, chemical, kappa_c/2 |grad c|^2, kappa_eta/2 |grad eta_i|^2 ...
 * The call queues one memset and one kernel on p->stream, copies the result out and returns after that stream has
 * drained. The sum is taken tile by tile in a fixed order: the same input gives the same bits on every run.
 * Limits: at most PF_STATIC_MAX_POINTS grid points (nx*ny*nz; 2048^2 and 256^3 fit, 512^3 does not) and n_eta <= 8;
 *   grid sizes as for pf_create. A grid beyond the limit is refused with PF_EUNSUPPORTED before anything is queued --
 *   use a context and pf_free_energy for those.
 * Sharing: there is one array per GPU, shared by every call in the process. It keeps the previous call's contents; the
 *   slots that must start at zero are cleared at the head of each call. Calls whose GPU work can overlap (two streams,
 *   two host threads) race on it and return garbage -- issue them on one stream or serialise them yourself.
 * First call on a device: looks up the device address of the array (cudaGetSymbolAddress, with that device current)
 *   and remembers it; make that first call during start-up, before any stream capture is begun.
 * PF_EINVAL: null pointers, bad ndim / n_eta / precision / dx, c or eta not device memory of the current device;
 * PF_EUNSUPPORTED: grid not a power of two in 16..2048 per axis, or more than PF_STATIC_MAX_POINTS points;
 * PF_ECUDA: no usable device or a CUDA call failed. */
#define PF_STATIC_TILE          4096                        /* grid points summed by one CTA                  */
#define PF_STATIC_MAX_POINTS    (1 << 24)                   /* 4096 tiles                                      */
#define PF_STATIC_SCRATCH_BYTES ((32 + 4096 * 10) * 8)      /* 327 936 bytes held per GPU for the process' life */
int pf_free_energy_static(const pf_params *p, const void *c, const void *eta, double *out);

/* Changes dt for subsequent steps (the dt sweep of the FS-vs-FD crossover); dt <= 0 -> PF_EINVAL. */
int pf_set_dt(pf_ctx *ctx, double dt);

/* Number of kernel launches (graph kernel nodes included) issued by this context so far. */
long long pf_launch_count(const pf_ctx *ctx);

/* Device time in milliseconds spent by kernel `which` of the most recent pf_step_fs call, measured
 * with CUDA events on the context's stream when profiling was switched on with pf_set_profiling
 * (which = 0 .. pf_num_fs_kernels()-1, in launch order within one step; averaged over the steps of
 * that call). Returns a negative value when unavailable. Profiling (on != 0) disables CUDA-graph replay and
 * programmatic dependent launch; the trajectory is the same. A single bracketed launch carries a few microseconds
 * of event overhead: for per-kernel figures without it use pf_launch_fs_kernel. */
int    pf_set_profiling(pf_ctx *ctx, int on);
/* Measured fp64 FMA rate of the current device in TFLOP/s (2 flops per FMA): a 20-line kernel of independent DFMA chains,
 * best of three timed launches. Diagnostic for the roofline notes (the Fourier-spectral kernels are
 * bound by fp64 issue and shared memory as much as by HBM). Synchronises the device. PF_EINVAL / PF_ECUDA on failure. */
int    pf_fp64_fma_peak(double *tflops);
/* Measured read rate of distributed shared memory on the current device: bytes per SM clock per SM that the CTAs of a
 * thread-block cluster of cluster_size CTAs (1, 2, 4, 8, 16) load from each other's shared memory with 16-byte loads
 * (remote != 0), or from their own through the same address path (remote == 0); one CTA per SM, the slowest CTA counts.
 * Diagnostic for DESIGN.md section 6 (why the 3D y/z passes are not merged inside a cluster; where the cluster-resident
 * small-grid kernel stops paying off). Allocates two small device buffers, synchronises the device.
 * PF_EINVAL: bad arguments; PF_EUNSUPPORTED: the device cannot run clusters of that size; PF_ENOMEM / PF_ECUDA. */
int    pf_dsmem_read_rate(int cluster_size, int remote, double *bytes_per_clk_per_sm);
int    pf_num_fs_kernels(const pf_ctx *ctx);
double pf_fs_kernel_ms(pf_ctx *ctx, int which);
const char *pf_fs_kernel_name(const pf_ctx *ctx, int which);

/* Timing aid: queues ONLY kernel `which` (0 .. pf_num_fs_kernels()-1) of one Fourier-spectral step on the context's
 * stream (asynchronous; launched as in a step, i.e. with programmatic stream serialization: its table-loading prologue may
 * overlap the tail of the launch before it, its reads and writes of the fields do not). A caller brackets a sequence of such calls -- e.g. the same kernel of several
 * contexts whose combined state exceeds the L2 -- with its own events. Needs fields (PF_ESTATE otherwise). Afterwards
 * the buffers are no trajectory: pf_step_*, pf_get_fields and pf_free_energy return PF_ESTATE until the next
 * pf_set_fields, further pf_launch_fs_kernel calls are allowed. */
int    pf_launch_fs_kernel(pf_ctx *ctx, int which);

const char *pf_strerror(int code);
const char *pf_last_cuda_error(const pf_ctx *ctx);      /* "" when none */

/* Frees everything the context owns (NULL is allowed). */
void pf_destroy(pf_ctx *ctx);

#ifdef __cplusplus
}
#endif
#endif
