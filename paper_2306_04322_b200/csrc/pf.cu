// pf.cu -- the C ABI of libpf (include/pf.h): context, buffers, tables, state tracking, launch
// sequences of the Fourier-spectral and finite-difference steps, CUDA-graph replay.
//
// Device data of a context (w = element size, N = nx*ny*nz, M = nx/2, F = 1 + n_eta):
//   real[2]  [F][nz][ny][nx]        real fields, double buffered (set/get, FD path)
//   zst      [F][nz][ny][M] complex "z-form" state of the spectral path (row_kernels.cu)
//   zg       [nz][ny][M]    complex z-form of g = df/dc
//   s2       [F][nz][ny][P2] complex, 3D only: (kx,ky)-spectral, z-real planes; s2[0] carries c between steps
//   g2       [nz][ny][P2]   complex, 3D only
//   park     [nz][ny][P2+16] complex scratch of the column kernels (dt M |xi|^2 g^ of the Cahn-Hilliard update)
//   tables   twiddles exp(-2 pi i k/n) for M, ny, nz, nx; |xi_d|^2 per axis (Eq. 16-21)
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include "../../include/pf.h"
#include "pf_kernels.cuh"

namespace pf {
void col2d_schedule(int nblk, int n_eta, int slots, int *grid_out, int *per_cta_out, std::vector<int> &sched);
void col2d_schedule_init(int nblk, int slots, int *grid_out, int *per_cta_out, std::vector<int> &sched);
}
using namespace pf;

namespace {

enum State { ST_NONE = 0, ST_REAL = 1, ST_SPECTRAL = 2, ST_BOTH = 3, ST_TIMING = 4 };
const int kMaxFsKernels = 6;
const int kProfBatch = 16;
const int kGraphSteps = 8;              // steps per captured graph (pf_step_fs calls of at least this many steps)

}  // namespace

struct pf_ctx {
    pf_params p;
    int F = 1, M = 0, P2 = 0;
    long N = 0;                          // grid points of ONE replica
    int B = 1;                           // replicas advanced together (pf_create_batch): further rows / planes / column blocks of the same launches
    int c2_nblk = 0;                     // column blocks per replica of the 2D last-axis kernel
    size_t w = 8;
    int device = 0;                      // the CUDA device the context was created on (every call checks it is current)
    cudaStream_t stream = nullptr;
    bool own_stream = false;
    bool graph_ok = true;
    bool use_wcol = false;              // -DPF_WCOL builds with PF_WCOL=1 in the environment: the persistent pipelined strided kernel (A/B runs, profiles/)
    void *real[2] = {nullptr, nullptr};
    int cur = 0;
    void *zst = nullptr, *zg = nullptr, *s2 = nullptr, *g2 = nullptr, *park = nullptr;
    void *tw_m = nullptr, *tw_y = nullptr, *tw_z = nullptr, *tw_nx = nullptr;
    void *kx2 = nullptr, *ky2 = nullptr, *kz2 = nullptr;
    double *acc = nullptr;
    int *queue = nullptr;               // work queue of the persistent strided kernel
    int state = ST_NONE;
    bool s2c_valid = false;
    // 2D: carried spectrum of c and the static schedule of the last-axis kernel (col2d_kernels.cu)
    bool park3d = false;                 // PF_COL3D_PARK=1: 3D z kernel re-transforms c every step (round-1 form, A/B runs)
    bool legacy_fd2d = false;            // PF_FD2D_LEGACY=1: fd_fused2d_kernel for every 2D shape (A/B runs)
    bool legacy_fd3d = false;            // PF_FD3D_LEGACY=1: fd_fused3d_kernel for every 3D shape (A/B runs)
    bool legacy_col2d = false;           // PF_COL2D_LEGACY=1: the one-CTA-per-(field, block) kernel of col_kernels.cu (A/B runs)
    void *carry = nullptr;
    bool carry_valid = false;
    int *c2_sched = nullptr, *c2_sched_init = nullptr, *c2_flags = nullptr;
    unsigned *c2_ticket = nullptr;       // place counter of the 2D last-axis kernel (nullptr with PF_COL2D_NOTICKET=1)
    int c2_grid = 0, c2_per = 0, c2_grid_init = 0, c2_per_init = 0;
    int sg_cs = 0;                       // > 0: cluster size of the resident small-grid kernel (sgrid_kernels.cu) serving this context
    int carveout = 0;                    // shared-memory carve-out both kernels of a 2D step run with (percent; 0: unset)
    TraceBuf *trace = nullptr;           // -DPF_TRACE builds only
    long long launches = 0;
    std::string cuda_err;
    // CUDA graph of one FS step
    cudaGraphExec_t fs_graph = nullptr;
    int fs_graph_nodes = 0;
    // profiling
    int profiling = 0;                   // events around every kernel of a step (no graph replay, no PDL)
    int nk = 0;
    const char *kname[kMaxFsKernels] = {};
    double kms[kMaxFsKernels] = {};
    std::vector<cudaEvent_t> pev;
};

namespace {

#define PF_CK(ctx, call)                                                      \
    do {                                                                      \
        cudaError_t e__ = (call);                                             \
        if (e__ != cudaSuccess) {                                             \
            (ctx)->cuda_err = std::string(#call) + ": " + cudaGetErrorString(e__); \
            return e__ == cudaErrorMemoryAllocation ? PF_ENOMEM : PF_ECUDA;   \
        }                                                                     \
    } while (0)

bool pow2_in_range(int n) { return n >= 16 && n <= 2048 && (n & (n - 1)) == 0; }

// squared frequency of one axis at index idx:
//   kind 0: xi^2, xi = 2 pi m / l, m = idx for idx <= n/2 else idx - n          (Eq. 16/19)
//   kind 1: 2 (1 - cos(dx xi)) / dx^2                                            (Eq. 17/20)
//   kind 2: (15 - 16 cos(dx xi) + cos(2 dx xi)) / (6 dx^2)                       (Eq. 18/21)
double axis_k2(int kind, int n, double dx, int idx)
{
    const double PI = 3.14159265358979323846264338327950288;
    const int m = (idx <= n / 2) ? idx : idx - n;
    const double xi = 2.0 * PI * (double)m / ((double)n * dx);
    if (kind == 0) return xi * xi;
    // dx*xi = 2 pi m / n: evaluate the cosine of the exact rational angle
    const double a = 2.0 * PI * (double)m / (double)n;
    if (kind == 1) return 2.0 * (1.0 - std::cos(a)) / (dx * dx);
    return (15.0 - 16.0 * std::cos(a) + std::cos(2.0 * a)) / (6.0 * dx * dx);
}

template <typename T> Model<T> make_model(const pf_params &p)
{
    Model<T> m;
    m.rho2 = (T)p.rho2; m.c_alpha = (T)p.c_alpha; m.c_beta = (T)p.c_beta; m.w = (T)p.w; m.alpha = (T)p.alpha;
    m.kappa_c = (T)p.kappa_c; m.kappa_eta = (T)p.kappa_eta;
    m.dt = (T)p.dt; m.M = (T)p.M; m.L = (T)p.L;
    m.dtM = (T)(p.dt * p.M); m.dtL = (T)(p.dt * p.L);
    m.dtMkc = (T)(p.dt * p.M * p.kappa_c); m.dtLke = (T)(p.dt * p.L * p.kappa_eta);
    m.gA0 = (T)(2.0 * p.rho2); m.gA1 = (T)(2.0 * p.rho2 * p.c_alpha); m.gA2 = (T)(2.0 * p.rho2 * (p.c_beta - p.c_alpha));
    m.eB0 = (T)(30.0 * p.rho2 * (p.c_beta * p.c_beta - p.c_alpha * p.c_alpha));
    m.eB1 = (T)(60.0 * p.rho2 * (p.c_beta - p.c_alpha));
    m.eW2 = (T)(2.0 * p.w); m.eW4a = (T)(4.0 * p.alpha * p.w);
    m.n_eta = p.n_eta;
    return m;
}

template <typename T> int upload_tables(pf_ctx *c)
{
    typedef typename V2<T>::type C;
    const long double PI = 3.141592653589793238462643383279502884L;
    auto twiddles = [&](int n, int count, void **dst) -> int {
        std::vector<C> h(count);
        for (int k = 0; k < count; ++k) {
            // reduce to the first octant for full accuracy at every k
            h[k].x = (T)cosl(2 * PI * (long double)k / n);
            h[k].y = (T)-sinl(2 * PI * (long double)k / n);
        }
        PF_CK(c, cudaMalloc(dst, sizeof(C) * count));
        PF_CK(c, cudaMemcpy(*dst, h.data(), sizeof(C) * count, cudaMemcpyHostToDevice));
        return PF_OK;
    };
    int rc;
    if ((rc = twiddles(c->M, c->M, &c->tw_m))) return rc;
    if ((rc = twiddles(c->p.n[1], c->p.n[1], &c->tw_y))) return rc;
    if ((rc = twiddles(c->p.n[2] > 1 ? c->p.n[2] : 2, c->p.n[2] > 1 ? c->p.n[2] : 2, &c->tw_z))) return rc;
    if ((rc = twiddles(c->p.n[0], c->M + 1, &c->tw_nx))) return rc;
    auto ktable = [&](int axis, int count, int padded, void **dst) -> int {
        std::vector<T> h(padded, (T)0);
        for (int k = 0; k < count; ++k) h[k] = (T)axis_k2(c->p.k2_kind, c->p.n[axis], c->p.dx[axis], k);
        PF_CK(c, cudaMalloc(dst, sizeof(T) * padded));
        PF_CK(c, cudaMemcpy(*dst, h.data(), sizeof(T) * padded, cudaMemcpyHostToDevice));
        return PF_OK;
    };
    if ((rc = ktable(0, c->M + 1, c->P2, &c->kx2))) return rc;
    if ((rc = ktable(1, c->p.n[1], c->p.n[1], &c->ky2))) return rc;
    if (c->p.ndim == 3) { if ((rc = ktable(2, c->p.n[2], c->p.n[2], &c->kz2))) return rc; }
    else {
        PF_CK(c, cudaMalloc(&c->kz2, sizeof(T) * 2));
        PF_CK(c, cudaMemset(c->kz2, 0, sizeof(T) * 2));
    }
    return PF_OK;
}

void drop_graph(pf_ctx *c)
{
    if (c->fs_graph) { cudaGraphExecDestroy(c->fs_graph); c->fs_graph = nullptr; }
}

// ---------------------------------------------------------------- launch sequences ----------------
template <typename T> RowParams<T> row_params(pf_ctx *c)
{
    typedef typename V2<T>::type C;
    RowParams<T> r{};                    // pdl = 0 unless the caller sets it
    r.zst = (C *)c->zst; r.zg = (C *)c->zg; r.real = (T *)c->real[c->cur];
    r.tw = (const C *)c->tw_m;
    r.zfs = c->B * (c->N / 2); r.rfs = c->B * c->N;   // replicas are further rows of every field
    r.nrows = c->p.n[1] * c->p.n[2] * c->B; r.F = c->F;
    r.carveout = c->carveout;
    r.m = make_model<T>(c->p);
#ifdef PF_TRACE
    r.trace = c->trace;
#endif
    return r;
}

template <typename T> ColParams<T> col_params(pf_ctx *c)
{
    typedef typename V2<T>::type C;
    ColParams<T> q;
    memset(&q, 0, sizeof(q));
    q.M = c->M; q.P2 = c->P2;
    q.twx = (const C *)c->tw_nx;
    q.kx2 = (const T *)c->kx2; q.ky2 = (const T *)c->ky2; q.kz2 = (const T *)c->kz2;
    q.acc = c->acc;
    q.queue = c->queue;
    q.park = (C *)c->park;
    q.m = make_model<T>(c->p);
#ifdef PF_TRACE
    q.trace = c->trace;
#endif
    return q;
}

template <typename T> Col2dParams<T> col2d_params(pf_ctx *c, bool init, bool pdl)
{
    typedef typename V2<T>::type C;
    Col2dParams<T> q;
    memset(&q, 0, sizeof(q));
    q.zst = (C *)c->zst; q.zg = (const C *)c->zg; q.carry = (C *)c->carry;
    q.zfs = c->B * (c->N / 2); q.M = c->M; q.nblk = c->c2_nblk;
    q.sched = init ? c->c2_sched_init : c->c2_sched;
    q.per_cta = init ? c->c2_per_init : c->c2_per;
    q.flags = c->c2_flags;
    q.ticket = c->c2_ticket;
    q.pdl = pdl;
    q.tw = (const C *)c->tw_y; q.twx = (const C *)c->tw_nx;
    q.kx2 = (const T *)c->kx2; q.ky2 = (const T *)c->ky2;
    q.m = make_model<T>(c->p);
#ifdef PF_TRACE
    q.trace = c->trace;
#endif
    return q;
}

struct KernelTimer {
    pf_ctx *c; int k = 0; cudaEvent_t *ev;
    KernelTimer(pf_ctx *ctx, cudaEvent_t *events) : c(ctx), ev(events) { if (ev) cudaEventRecord(ev[0], c->stream); }
    void mark(const char *name)
    {
        if (k < kMaxFsKernels) { c->kname[k] = name; if (ev) cudaEventRecord(ev[k + 1], c->stream); ++k; }
    }
};

// 3D: (kx,ky)-spectral planes of z-form arrays: dst slot s <- FFT_y(unpack(src slot s)); with galt, slot 0 is zg -> g2
template <typename T> cudaError_t mid_forward(pf_ctx *c, const void *zsrc, long zfs, void *dst, long dfs, int nslots,
                                              bool galt, bool pdl)
{
    typedef typename V2<T>::type C;
    const int ny = c->p.n[1], nz = c->p.n[2];
    ColParams<T> q = col_params<T>(c);
    q.in0 = (const C *)zsrc; q.in_fs = zfs; q.in_rs = c->M; q.in_bs = (long)ny * c->M;
    q.out = (C *)dst; q.out_fs = dfs; q.out_rs = c->P2; q.out_bs = (long)ny * c->P2;
    if (galt) { q.alt_in = (const C *)c->zg; q.alt_out = (C *)c->g2; }
    q.tw = (const C *)c->tw_y;
    q.pdl = pdl;
    ++c->launches;
    return launch_col<T>(COL_3D_MIDFWD, ny, nslots, nz * c->B, q, c->stream);    // replicas are further planes
}

// One FS step. 2D: x kernel, y kernel. 3D: x kernel, y-forward, z kernel, y-inverse. All launched with programmatic
// stream serialization: each kernel's prologue overlaps its predecessor's tail (griddepcontrol in the kernels).
// events != nullptr: one event after every kernel (profiling; launches are then kept strictly serial).
// only >= 0: launch just that kernel of the step (timing aid, pf_launch_fs_kernel), with the same launch attribute as in a step.
template <typename T> int fs_one_step(pf_ctx *c, cudaEvent_t *events, int only = -1)
{
    typedef typename V2<T>::type C;
    const int ny = c->p.n[1], nz = c->p.n[2];
    const long zfs = c->B * (c->N / 2);
    const bool pdl = events == nullptr;
    KernelTimer kt(c, events);
    auto want = [&](int k) { return only < 0 || only == k; };
    if (want(0)) {
        RowParams<T> r = row_params<T>(c);
        r.pdl = pdl;
        PF_CK(c, launch_row<T>(ROW_STEP, c->p.n[0], r, c->stream)); ++c->launches;
    }
    kt.mark("row_c2r_nonlinear_r2c");
    C *zst = (C *)c->zst;
    if (c->p.ndim == 2) {
        if (want(1)) {
            ColParams<T> q = col_params<T>(c);
            q.tw = (const C *)c->tw_y;
            q.in_rs = q.out_rs = c->M;
            q.in0 = zst; q.in1 = (const C *)c->zg; q.out = zst; q.in_fs = q.out_fs = zfs;
            q.has_c = 1; q.pdl = pdl;
            cudaError_t e = cudaErrorNotSupported;
#ifdef PF_WCOL
            if (c->use_wcol) e = launch_wcol2d<T>(ny, c->F, q, c->stream);
            else
#endif
            if (!c->legacy_col2d) e = launch_col2d<T>(ny, col2d_params<T>(c, false, pdl), c->c2_grid, c->stream);
            if (e == cudaErrorNotSupported) e = launch_col<T>(COL_2D_LAST, ny, c->F, 1, q, c->stream);
            PF_CK(c, e); ++c->launches;
        }
        kt.mark("col_y_fft_update_ifft");
    } else {
        const long s2rs = (long)nz * ny * c->P2;               // one replica of one field
        const long s2fs = s2rs * c->B;
        C *s2 = (C *)c->s2;
        if (want(1)) PF_CK(c, mid_forward<T>(c, zst, zfs, s2, s2fs, c->F, true, pdl));
        kt.mark("col_y_fwd");
        if (want(2)) {
            ColParams<T> q = col_params<T>(c);
            q.tw = (const C *)c->tw_z;
            q.in_rs = q.out_rs = (long)ny * c->P2; q.ncols = ny * c->P2;
            q.in0 = s2; q.in1 = (const C *)c->g2; q.out = s2; q.in_fs = q.out_fs = s2fs;
            q.in_bs = q.out_bs = s2rs;                         // blockIdx.y = replica
            q.has_c = c->park3d ? 1 : 2; q.pdl = pdl;          // 2: c^ carried in `park` (filled by to_spectral)
            PF_CK(c, launch_col<T>(COL_3D_LAST, nz, c->F, c->B, q, c->stream)); ++c->launches;
        }
        kt.mark("col_z_fft_update_ifft");
        if (want(3)) {
            ColParams<T> v = col_params<T>(c);
            v.tw = (const C *)c->tw_y;
            v.in0 = s2; v.in_fs = s2fs; v.in_rs = c->P2; v.in_bs = (long)ny * c->P2;
            v.out = zst; v.out_fs = zfs; v.out_rs = c->M; v.out_bs = (long)ny * c->M;
            v.pdl = pdl;
            PF_CK(c, launch_col<T>(COL_3D_MIDINV, ny, c->F, nz * c->B, v, c->stream)); ++c->launches;
        }
        kt.mark("col_y_inv");
    }
    c->nk = kt.k;
    return PF_OK;
}

// real fields -> z-form state (and, in 3D, the carried (kx,ky)-spectral planes of c)
template <typename T> int to_spectral(pf_ctx *c, bool need_carry = true)
{
    if (c->state == ST_REAL) {
        RowParams<T> r = row_params<T>(c);
        PF_CK(c, launch_row<T>(ROW_SET, c->p.n[0], r, c->stream)); ++c->launches;
        c->state = ST_BOTH;
    }
    if (c->p.ndim == 2 && c->carry && !c->carry_valid && need_carry) {
        PF_CK(c, launch_col2d<T>(c->p.n[1], col2d_params<T>(c, true, false), c->c2_grid_init, c->stream)); ++c->launches;
        c->carry_valid = true;
    }
    if (c->p.ndim == 3 && !c->s2c_valid) {
        typedef typename V2<T>::type C;
        PF_CK(c, mid_forward<T>(c, c->zst, 0, c->s2, 0, 1, false, false));
        if (!c->park3d) {
            // the carried spectrum c^ of the z kernel, in its thread-linear order (same launch geometry, slot 0 only)
            const int ny = c->p.n[1], nz = c->p.n[2];
            ColParams<T> q = col_params<T>(c);
            q.tw = (const C *)c->tw_z;
            q.in_rs = q.out_rs = (long)ny * c->P2; q.ncols = ny * c->P2;
            q.in0 = (const C *)c->s2; q.in1 = (const C *)c->g2; q.out = (C *)c->s2;
            q.in_fs = q.out_fs = (long)nz * ny * c->P2 * c->B;
            q.in_bs = q.out_bs = (long)nz * ny * c->P2;
            q.has_c = 3; q.pdl = 0;
            PF_CK(c, launch_col<T>(COL_3D_LAST, nz, 1, c->B, q, c->stream)); ++c->launches;
        }
        c->s2c_valid = true;
    }
    return PF_OK;
}

template <typename T> int to_real(pf_ctx *c)
{
    if (c->state == ST_SPECTRAL) {
        RowParams<T> r = row_params<T>(c);
        PF_CK(c, launch_row<T>(ROW_GET, c->p.n[0], r, c->stream)); ++c->launches;
        c->state = ST_BOTH;
    }
    return PF_OK;
}

// small square 2D grids: every step of the call inside ONE launch, state resident in a cluster's shared memory
template <typename T> int resident_steps(pf_ctx *c, int nsteps)
{
    typedef typename V2<T>::type C;
    int rc = to_spectral<T>(c, false);
    if (rc) return rc;
    SgParams<T> q;
    q.zst = (C *)c->zst; q.zfs = c->B * (c->N / 2); q.F = c->F; q.nsteps = nsteps;
    q.tw_m = (const C *)c->tw_m; q.tw_y = (const C *)c->tw_y; q.twx = (const C *)c->tw_nx;
    q.kx2 = (const T *)c->kx2; q.ky2 = (const T *)c->ky2;
    q.m = make_model<T>(c->p);
    PF_CK(c, launch_sgrid<T>(c->p.n[0], c->p.n[1], q, c->sg_cs, c->B, c->stream)); ++c->launches;
    c->carry_valid = false;              // the kernel keeps its own copy of c^; the carried spectrum in global memory is stale now
    c->state = ST_SPECTRAL;
    return PF_OK;
}

template <typename T> int step_fs(pf_ctx *c, int nsteps)
{
    // one launch of the resident kernel costs about 6.5 us + 4.7 us per step at 64^2, two launches per step 9 us per step
    if (c->sg_cs > 0 && !c->profiling && nsteps >= 2) return resident_steps<T>(c, nsteps);
    int rc = to_spectral<T>(c);
    if (rc) return rc;
    if (c->profiling) {
        // events around every kernel; a batch of steps is queued before the host waits, so launch latency stays hidden
        const int B = kProfBatch, per = kMaxFsKernels + 1;
        if (c->pev.empty()) {
            c->pev.resize((size_t)B * per);
            for (auto &e : c->pev) PF_CK(c, cudaEventCreate(&e));
        }
        double sum[kMaxFsKernels] = {};
        for (int s0 = 0; s0 < nsteps; s0 += B) {
            const int nb = (nsteps - s0 < B) ? nsteps - s0 : B;
            for (int s = 0; s < nb; ++s)
                if ((rc = fs_one_step<T>(c, c->pev.data() + (size_t)s * per))) return rc;
            PF_CK(c, cudaStreamSynchronize(c->stream));
            for (int s = 0; s < nb; ++s)
                for (int k = 0; k < c->nk; ++k) {
                    float ms = 0;
                    cudaEventElapsedTime(&ms, c->pev[(size_t)s * per + k], c->pev[(size_t)s * per + k + 1]);
                    sum[k] += ms;
                }
        }
        for (int k = 0; k < c->nk; ++k) c->kms[k] = sum[k] / nsteps;
    } else {
        // Every kernel is launched with programmatic stream serialization, so a kernel's CTAs become resident under its
        // predecessor's last CTAs. Long runs replay a captured graph of kGraphSteps steps (the programmatic edges between
        // ALL its kernels are kept; a graph of one step would serialise at every step boundary: 2.9 us of 52 at 1024^2,
        // DESIGN.md section 2); what is left, and short calls, are plain launches.
        if (!c->fs_graph && c->graph_ok && nsteps >= kGraphSteps) {
            cudaGraph_t g = nullptr;
            const long long before = c->launches;
            if (cudaStreamBeginCapture(c->stream, cudaStreamCaptureModeThreadLocal) == cudaSuccess) {
                for (int s = 0; s < kGraphSteps && !rc; ++s) rc = fs_one_step<T>(c, nullptr);
                cudaError_t e = cudaStreamEndCapture(c->stream, &g);
                c->fs_graph_nodes = (int)(c->launches - before);
                c->launches = before;
                if (rc) { if (g) cudaGraphDestroy(g); return rc; }
                PF_CK(c, e);
                e = cudaGraphInstantiate(&c->fs_graph, g, 0);
                cudaGraphDestroy(g);
                PF_CK(c, e);
            } else {
                cudaGetLastError();          // a stream that cannot be captured: plain launches
                c->graph_ok = false;
            }
        }
        int left = nsteps;
        for (; c->fs_graph && left >= kGraphSteps; left -= kGraphSteps) {
            PF_CK(c, cudaGraphLaunch(c->fs_graph, c->stream));
            c->launches += c->fs_graph_nodes;
        }
        for (; left > 0; --left)
            if ((rc = fs_one_step<T>(c, nullptr))) return rc;
    }
    c->state = ST_SPECTRAL;
    return PF_OK;
}

template <typename T> int step_fd(pf_ctx *c, int nsteps)
{
    int rc = to_real<T>(c);
    if (rc) return rc;
    FdParams<T> f;
    f.nx = c->p.n[0]; f.ny = c->p.n[1]; f.nz = c->p.n[2]; f.N = c->N; f.fs = c->B * c->N; f.nbatch = c->B;
    for (int d = 0; d < 3; ++d) f.rdx2[d] = (d < c->p.ndim) ? (T)(1.0 / (c->p.dx[d] * c->p.dx[d])) : (T)0;
    f.m = make_model<T>(c->p);
    for (int s = 0; s < nsteps; ++s) {
        T *cu = (T *)c->real[c->cur], *nw = (T *)c->real[c->cur ^ 1];
        f.c = cu; f.eta = cu + c->B * c->N; f.c_new = nw; f.eta_new = nw + c->B * c->N;
        if (c->p.ndim == 2) {
            cudaError_t e = c->legacy_fd2d ? cudaErrorNotSupported : launch_fd2d_pair<T>(f, c->stream);
            if (e == cudaErrorNotSupported) e = launch_fd_fused2d<T>(f, c->stream);
            PF_CK(c, e);
            c->launches += 1;
        } else {
            for (int b = 0; b < c->B; ++b) {             // 3D: one launch per replica (the z chunks take blockIdx.z)
                FdParams<T> g = f;
                g.nbatch = 1;
                g.c += (long)b * c->N; g.eta += (long)b * c->N; g.c_new += (long)b * c->N; g.eta_new += (long)b * c->N;
                cudaError_t e = c->legacy_fd3d ? cudaErrorNotSupported : launch_fd3d_march<T>(g, c->stream);
                if (e == cudaErrorNotSupported) e = launch_fd_fused3d<T>(g, c->stream);
                PF_CK(c, e);
                c->launches += 1;
            }
        }
        c->cur ^= 1;
    }
    c->state = ST_REAL;
    c->s2c_valid = false;
    c->carry_valid = false;
    return PF_OK;
}

template <typename T> int free_energy(pf_ctx *c, int kind, double *out)
{
    typedef typename V2<T>::type C;
    int rc = to_real<T>(c);
    if (rc) return rc;
    const int p = c->p.n_eta, nacc = 2 + p;
    PF_CK(c, cudaMemsetAsync(c->acc, 0, sizeof(double) * 32, c->stream));
    EnergyParams<T> e;
    e.c = (const T *)c->real[c->cur]; e.eta = e.c + c->N;
    e.nx = c->p.n[0]; e.ny = c->p.n[1]; e.nz = c->p.n[2]; e.N = c->N;
    for (int d = 0; d < 3; ++d) e.rdx[d] = (d < c->p.ndim) ? (T)(1.0 / c->p.dx[d]) : (T)0;
    e.gradient_kind = kind; e.acc = c->acc; e.m = make_model<T>(c->p);
    PF_CK(c, launch_energy<T>(e, c->stream)); ++c->launches;
    double scale_grad = 1.0;
    if (kind == 0) {
        // Parseval: sum_x |grad u|^2 = (1/N) sum_k |xi|^2 |u^_k|^2
        if ((rc = to_spectral<T>(c))) return rc;
        ColParams<T> q = col_params<T>(c);
        q.acc = c->acc + 1;
        const int ny = c->p.n[1], nz = c->p.n[2];
        if (c->p.ndim == 2) {
            q.tw = (const C *)c->tw_y; q.in0 = (const C *)c->zst; q.in_fs = c->N / 2; q.in_rs = c->M;
            PF_CK(c, launch_col<T>(COL_2D_ENERGY, ny, c->F, 1, q, c->stream)); ++c->launches;
        } else {
            const long s2fs = (long)nz * ny * c->P2;
            if (p > 0) PF_CK(c, mid_forward<T>(c, (C *)c->zst + c->N / 2, c->N / 2, (C *)c->s2 + s2fs, s2fs, p, false, false));
            q.tw = (const C *)c->tw_z; q.in0 = (const C *)c->s2; q.in_fs = s2fs; q.in_rs = (long)ny * c->P2;
            q.ncols = ny * c->P2;
            PF_CK(c, launch_col<T>(COL_3D_ENERGY, nz, c->F, 1, q, c->stream)); ++c->launches;
        }
        scale_grad = 1.0 / (double)c->N;
    }
    double h[32];
    PF_CK(c, cudaMemcpyAsync(h, c->acc, sizeof(double) * nacc, cudaMemcpyDeviceToHost, c->stream));
    PF_CK(c, cudaStreamSynchronize(c->stream));
    double dV = 1.0;
    for (int d = 0; d < c->p.ndim; ++d) dV *= c->p.dx[d];
    out[1] = h[0] * dV;
    out[2] = 0.5 * c->p.kappa_c * h[1] * scale_grad * dV;
    double tot = out[1] + out[2];
    for (int k = 0; k < p; ++k) { out[3 + k] = 0.5 * c->p.kappa_eta * h[2 + k] * scale_grad * dV; tot += out[3 + k]; }
    out[0] = tot;
    return PF_OK;
}

// every entry point runs on the device the context was created on; a different current device is a caller error
bool on_device(const pf_ctx *c)
{
    int d = -1;
    return cudaGetDevice(&d) == cudaSuccess && d == c->device;
}

// Fields between the caller's arrays and real[]. Caller: c [B][N], eta [B][p][N] (replica-major); library: [F][B][N]
// (a replica is a run of rows of every field). to_lib: caller -> library, else library -> caller.
int copy_fields(pf_ctx *c, void *user_c, void *user_eta, void *lib, bool to_lib, cudaMemcpyKind kind)
{
    const size_t fb = (size_t)c->N * c->w;               // one field of one replica
    char *lc = (char *)lib, *le = lc + fb * c->B;
    const int p = c->p.n_eta;
    if (to_lib) PF_CK(c, cudaMemcpyAsync(lc, user_c, fb * c->B, kind, c->stream));
    else PF_CK(c, cudaMemcpyAsync(user_c, lc, fb * c->B, kind, c->stream));
    if (p == 0) return PF_OK;
    if (c->B == 1) {
        if (to_lib) PF_CK(c, cudaMemcpyAsync(le, user_eta, fb * p, kind, c->stream));
        else PF_CK(c, cudaMemcpyAsync(user_eta, le, fb * p, kind, c->stream));
        return PF_OK;
    }
    for (int f = 0; f < p; ++f) {                        // B runs of N elements: pitch p*N on the caller's side, N on ours
        char *ue = (char *)user_eta + fb * f, *lf = le + fb * c->B * f;
        if (to_lib) PF_CK(c, cudaMemcpy2DAsync(lf, fb, ue, fb * p, fb, c->B, kind, c->stream));
        else PF_CK(c, cudaMemcpy2DAsync(ue, fb * p, lf, fb, fb, c->B, kind, c->stream));
    }
    return PF_OK;
}

}  // namespace

// fp64 FMA rate of the device (pf_fp64_fma_peak): 8 independent DFMA chains per thread, 1024 threads per CTA, 4 CTAs per SM
__global__ void __launch_bounds__(1024) fp64_peak_kernel(double *out, int iters, double a, double b)
{
    double x[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) x[i] = 1.0 + 1e-9 * (threadIdx.x + i);
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 8; ++i) x[i] = fma(x[i], a, b);
    }
    double sum = 0.0;
#pragma unroll
    for (int i = 0; i < 8; ++i) sum += x[i];
    if (sum == 12345.678) out[0] = sum;            // never true: keeps the chains alive
}

// ================================================================== C ABI =========================
extern "C" {

const char *pf_strerror(int code)
{
    switch (code) {
    case PF_OK: return "ok";
    case PF_EINVAL: return "invalid argument";
    case PF_ENOMEM: return "out of device memory";
    case PF_ECUDA: return "CUDA error";
    case PF_ESTATE: return "no fields set";
    case PF_EUNSUPPORTED: return "unsupported configuration (grid size, or a feature this kind of context does not have)";
    }
    return "unknown error";
}

const char *pf_last_cuda_error(const pf_ctx *ctx) { return ctx ? ctx->cuda_err.c_str() : ""; }

void pf_destroy(pf_ctx *c)
{
    if (!c) return;
    drop_graph(c);
#ifdef PF_TRACE
    if (c->trace) {
        cudaDeviceSynchronize();
        const char *fn = getenv("PF_TRACE_FILE");
        if (FILE *fh = fn ? fopen(fn, "a") : nullptr) {
            const unsigned long long n = c->trace->n < c->trace->cap ? c->trace->n : c->trace->cap;
            for (unsigned long long i = 0; i < n; ++i)
                fprintf(fh, "%llu %llu %llu %llu\n", c->trace->rec[3 * i] >> 32, c->trace->rec[3 * i] & 0xffffffffull,
                        c->trace->rec[3 * i + 1], c->trace->rec[3 * i + 2]);
            fclose(fh);
        }
        cudaFree(c->trace);
    }
#endif
    for (auto &e : c->pev) if (e) cudaEventDestroy(e);
    void *bufs[] = {c->real[0], c->real[1], c->zst, c->zg, c->s2, c->g2, c->park, c->tw_m, c->tw_y, c->tw_z,
                    c->tw_nx, c->kx2, c->ky2, c->kz2, c->acc, c->queue, c->carry, c->c2_sched, c->c2_sched_init,
                    c->c2_flags, c->c2_ticket};
    for (void *b : bufs) if (b) cudaFree(b);
    if (c->own_stream) cudaStreamDestroy(c->stream);
    delete c;
}

static int create_impl(const pf_params *p, int nbatch, pf_ctx **out)
{
    if (!p || !out) return PF_EINVAL;
    if (nbatch < 1 || nbatch > 4096) return PF_EINVAL;
    if (p->ndim != 2 && p->ndim != 3) return PF_EINVAL;
    if (p->n_eta < 0 || p->n_eta > 8) return PF_EINVAL;
    if (!(p->dt > 0.0)) return PF_EINVAL;
    if (p->precision != PF_F32 && p->precision != PF_F64) return PF_EINVAL;
    if (p->k2_kind < 0 || p->k2_kind > 2) return PF_EINVAL;
    for (int d = 0; d < p->ndim; ++d) if (!(p->dx[d] > 0.0)) return PF_EINVAL;
    for (int d = 0; d < p->ndim; ++d) if (!pow2_in_range(p->n[d])) return PF_EUNSUPPORTED;
    if (p->ndim == 2 && p->n[2] != 1) return PF_EUNSUPPORTED;
    if (p->ndim == 3 && (long)p->n[2] * nbatch > 65535) return PF_EUNSUPPORTED;      // planes of all replicas = blockIdx.y of the y kernels

    int ndev = 0, dev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev <= 0) { cudaGetLastError(); return PF_ECUDA; }
    if (cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); return PF_ECUDA; }

    pf_ctx *c = new (std::nothrow) pf_ctx();
    if (!c) return PF_ENOMEM;
    c->p = *p;
    c->B = nbatch;
    c->device = dev;
#ifdef PF_WCOL                       // the measured-slower persistent strided kernel is compiled into ablation builds only
    { const char *e = getenv("PF_WCOL"); c->use_wcol = (e && e[0] == '1' && nbatch == 1); }
#endif
    { const char *e = getenv("PF_COL2D_LEGACY"); c->legacy_col2d = (e && e[0] == '1' && nbatch == 1); }
    { const char *e = getenv("PF_COL3D_PARK"); c->park3d = (e && e[0] == '1'); }
    { const char *e = getenv("PF_FD2D_LEGACY"); c->legacy_fd2d = (e && e[0] == '1'); }
    { const char *e = getenv("PF_FD3D_LEGACY"); c->legacy_fd3d = (e && e[0] == '1'); }
    { const char *e = getenv("PF_NO_GRAPH"); if (e && e[0] == '1') c->graph_ok = false; }
    if (p->ndim == 2) { c->p.n[2] = 1; c->p.dx[2] = 1.0; }
    c->F = 1 + p->n_eta;
    c->M = p->n[0] / 2;
    c->P2 = ((c->M + 1 + 15) / 16) * 16;
    c->N = (long)c->p.n[0] * c->p.n[1] * c->p.n[2];
    c->w = (p->precision == PF_F64) ? 8 : 4;
    c->stream = (cudaStream_t)p->stream;
    if (!c->stream) {
        // NULL: a private blocking stream (ordered with the legacy default stream, and capturable)
        if (cudaStreamCreate(&c->stream) != cudaSuccess) { cudaGetLastError(); delete c; return PF_ECUDA; }
        c->own_stream = true;
    }

    auto fail = [&](int rc) { pf_destroy(c); return rc; };
    auto alloc = [&](void **dst, size_t bytes) -> int {
        cudaError_t e = cudaMalloc(dst, bytes);
        if (e != cudaSuccess) { cudaGetLastError(); return e == cudaErrorMemoryAllocation ? PF_ENOMEM : PF_ECUDA; }
        e = cudaMemset(*dst, 0, bytes);
        return e == cudaSuccess ? PF_OK : PF_ECUDA;
    };
    const size_t fb = (size_t)c->N * c->w * c->B;          // one real field of every replica
    int rc;
    if ((rc = alloc(&c->real[0], fb * c->F)) || (rc = alloc(&c->real[1], fb * c->F)) ||
        (rc = alloc(&c->zst, fb * c->F)) || (rc = alloc(&c->zg, fb)) ||
        (rc = alloc((void **)&c->acc, sizeof(double) * 32)) || (rc = alloc((void **)&c->queue, sizeof(int) * 4)) ||
        (rc = alloc(&c->park, (size_t)(c->P2 + 16) * c->p.n[1] * c->p.n[2] * 2 * c->w * c->B)))
        return fail(rc);
    if (p->ndim == 3) {
        const size_t pb = (size_t)c->p.n[2] * c->p.n[1] * c->P2 * 2 * c->w * c->B;
        if ((rc = alloc(&c->s2, pb * c->F)) || (rc = alloc(&c->g2, pb))) return fail(rc);
    }
    rc = (p->precision == PF_F64) ? upload_tables<double>(c) : upload_tables<float>(c);
    if (rc) return fail(rc);
    if (p->ndim == 2 && !c->legacy_col2d && !c->use_wcol) {
        Col2dShapeInfo si;
        cudaError_t e = (p->precision == PF_F64) ? col2d_shape<double>(c->p.n[1], c->M, &si) : col2d_shape<float>(c->p.n[1], c->M, &si);
        if (e != cudaSuccess) { c->cuda_err = cudaGetErrorString(e); cudaGetLastError(); return fail(PF_ECUDA); }
        c->carveout = si.carveout_pct;
        c->c2_nblk = si.nblk;
        const int nblk_all = si.nblk * c->B;               // the replicas' column blocks are dealt out together
        std::vector<int> sched, sched_init;
        col2d_schedule(nblk_all, p->n_eta, si.slots, &c->c2_grid, &c->c2_per, sched);
        col2d_schedule_init(nblk_all, si.slots, &c->c2_grid_init, &c->c2_per_init, sched_init);
        if ((rc = alloc(&c->carry, (size_t)si.carry_elems * c->B * 2 * c->w)) ||
            (rc = alloc((void **)&c->c2_sched, sizeof(int) * sched.size())) ||
            (rc = alloc((void **)&c->c2_sched_init, sizeof(int) * sched_init.size())) ||
            (rc = alloc((void **)&c->c2_flags, sizeof(int) * (size_t)nblk_all)))
            return fail(rc);
        { const char *e = getenv("PF_COL2D_NOTICKET");
          if (!(e && e[0] == '1') && (rc = alloc((void **)&c->c2_ticket, 64))) return fail(rc); }
        if (cudaMemcpy(c->c2_sched, sched.data(), sizeof(int) * sched.size(), cudaMemcpyHostToDevice) != cudaSuccess ||
            cudaMemcpy(c->c2_sched_init, sched_init.data(), sizeof(int) * sched_init.size(), cudaMemcpyHostToDevice) != cudaSuccess) {
            cudaGetLastError();
            return fail(PF_ECUDA);
        }
    }
    if (p->ndim == 2) {
        // Square grids up to 64^2 run pf_step_fs in the cluster-resident kernel (sgrid_kernels.cu): 64^2, c + 2 eta, fp64:
        // 4.7 us per step against 11.0 us on the two-kernel path; at 128^2 the two paths are level and the two-kernel path
        // stays (profiles/r2_small_grids.md). A single simulation takes a cluster of 16 CTAs, a batch as many CTAs per
        // replica as keep the whole batch on the machine at once.
        // PF_RESIDENT=0: two-kernel path for every size (A/B runs); PF_SG_CLUSTER=<n>: resident path with clusters of >= n
        // CTAs for every size that sgrid_kernels.cu serves and that fits.
        const char *er = getenv("PF_RESIDENT"), *ec = getenv("PF_SG_CLUSTER");
        if (!(er && er[0] == '0') && (ec || (p->n[0] == p->n[1] && p->n[0] <= 64))) {
            int sms = 148;
            cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
            int want = ec ? atoi(ec) : (c->B > 1 ? sms / c->B : 16);
            if (want < 1) want = 1;
            if (want > 16) want = 16;
            while (want & (want - 1)) want &= want - 1;
            c->sg_cs = (p->precision == PF_F64) ? sgrid_plan<double>(p->n[0], p->n[1], c->F, want)
                                                : sgrid_plan<float>(p->n[0], p->n[1], c->F, want);
            cudaGetLastError();
        }
    }
#ifdef PF_TRACE
    if (getenv("PF_TRACE_FILE")) {
        const unsigned long long cap = 1ull << 20;
        if (cudaMallocManaged((void **)&c->trace, sizeof(TraceBuf) + 3 * cap * sizeof(unsigned long long)) == cudaSuccess) {
            c->trace->n = 0; c->trace->cap = cap;
        } else { cudaGetLastError(); c->trace = nullptr; }
    }
#endif
    *out = c;
    return PF_OK;
}

int pf_create(const pf_params *p, pf_ctx **out) { return create_impl(p, 1, out); }
int pf_create_batch(const pf_params *p, int nbatch, pf_ctx **out) { return create_impl(p, nbatch, out); }
int pf_batch_size(const pf_ctx *c) { return c ? c->B : 0; }

int pf_set_fields(pf_ctx *c, const void *fc, const void *eta, int where)
{
    if (!c || !fc || (c->p.n_eta > 0 && !eta)) return PF_EINVAL;
    if (where != PF_HOST && where != PF_DEVICE) return PF_EINVAL;
    if (!on_device(c)) return PF_EINVAL;
    int rc = copy_fields(c, const_cast<void *>(fc), const_cast<void *>(eta), c->real[c->cur], true,
                         where == PF_HOST ? cudaMemcpyHostToDevice : cudaMemcpyDeviceToDevice);
    if (rc) return rc;
    if (where == PF_HOST) PF_CK(c, cudaStreamSynchronize(c->stream));
    c->state = ST_REAL;
    c->s2c_valid = false;
    c->carry_valid = false;
    return PF_OK;
}

int pf_get_fields(pf_ctx *c, void *fc, void *eta, int where)
{
    if (!c || !fc || (c->p.n_eta > 0 && !eta)) return PF_EINVAL;
    if (where != PF_HOST && where != PF_DEVICE) return PF_EINVAL;
    if (!on_device(c)) return PF_EINVAL;
    if (c->state == ST_NONE || c->state == ST_TIMING) return PF_ESTATE;
    int rc = (c->p.precision == PF_F64) ? to_real<double>(c) : to_real<float>(c);
    if (rc) return rc;
    rc = copy_fields(c, fc, eta, c->real[c->cur], false,
                     where == PF_HOST ? cudaMemcpyDeviceToHost : cudaMemcpyDeviceToDevice);
    if (rc) return rc;
    if (where == PF_HOST) PF_CK(c, cudaStreamSynchronize(c->stream));
    return PF_OK;
}

int pf_step_fs(pf_ctx *c, int nsteps)
{
    if (!c || nsteps < 0) return PF_EINVAL;
    if (nsteps == 0) return PF_OK;
    if (!on_device(c)) return PF_EINVAL;
    if (c->state == ST_NONE || c->state == ST_TIMING) return PF_ESTATE;
    return (c->p.precision == PF_F64) ? step_fs<double>(c, nsteps) : step_fs<float>(c, nsteps);
}

int pf_step_fd(pf_ctx *c, int nsteps)
{
    if (!c || nsteps < 0) return PF_EINVAL;
    if (nsteps == 0) return PF_OK;
    if (!on_device(c)) return PF_EINVAL;
    if (c->state == ST_NONE || c->state == ST_TIMING) return PF_ESTATE;
    return (c->p.precision == PF_F64) ? step_fd<double>(c, nsteps) : step_fd<float>(c, nsteps);
}

int pf_free_energy(pf_ctx *c, int gradient_kind, double *out)
{
    if (!c || !out || (gradient_kind != 0 && gradient_kind != 1)) return PF_EINVAL;
    if (!on_device(c)) return PF_EINVAL;
    if (c->B > 1) return PF_EUNSUPPORTED;              /* one replica at a time: read the fields out */
    if (c->state == ST_NONE || c->state == ST_TIMING) return PF_ESTATE;
    return (c->p.precision == PF_F64) ? free_energy<double>(c, gradient_kind, out)
                                      : free_energy<float>(c, gradient_kind, out);
}

int pf_set_dt(pf_ctx *c, double dt)
{
    if (!c || !(dt > 0.0)) return PF_EINVAL;
    c->p.dt = dt;
    drop_graph(c);                       // dt is baked into the captured kernel arguments
    return PF_OK;
}

long long pf_launch_count(const pf_ctx *c) { return c ? c->launches : 0; }

int pf_fp64_fma_peak(double *tflops)
{
    if (!tflops) return PF_EINVAL;
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) {
        cudaGetLastError();
        return PF_ECUDA;
    }
    double *buf = nullptr;
    cudaEvent_t e0, e1;
    if (cudaMalloc((void **)&buf, 64) != cudaSuccess) { cudaGetLastError(); return PF_ECUDA; }
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    const int iters = 1 << 14, grid = sms * 4;
    double best = 0.0;
    for (int rep = 0; rep < 4; ++rep) {                  // first pass is the warm-up
        cudaEventRecord(e0);
        fp64_peak_kernel<<<grid, 1024>>>(buf, iters, 0.999999, 1e-6);
        cudaEventRecord(e1);
        if (cudaEventSynchronize(e1) != cudaSuccess) { cudaGetLastError(); cudaFree(buf); return PF_ECUDA; }
        float ms = 0;
        cudaEventElapsedTime(&ms, e0, e1);
        const double t = 2.0 * 8.0 * iters * 1024.0 * grid / (ms * 1e-3) / 1e12;
        if (rep > 0 && t > best) best = t;
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(buf);
    *tflops = best;
    return PF_OK;
}

int pf_set_profiling(pf_ctx *c, int on)
{
    if (!c) return PF_EINVAL;
    c->profiling = on > 0 ? 1 : 0;
    for (double &v : c->kms) v = -1.0;
    return PF_OK;
}
int pf_launch_fs_kernel(pf_ctx *c, int which)
{
    if (!c || which < 0 || which >= pf_num_fs_kernels(c)) return PF_EINVAL;
    if (!on_device(c)) return PF_EINVAL;
    if (c->state == ST_NONE) return PF_ESTATE;   /* ST_TIMING is fine here */
    int rc = (c->p.precision == PF_F64) ? to_spectral<double>(c) : to_spectral<float>(c);
    if (rc) return rc;
    rc = (c->p.precision == PF_F64) ? fs_one_step<double>(c, nullptr, which) : fs_one_step<float>(c, nullptr, which);
    // one kernel of a step applied on its own: the buffers are no trajectory any more. The context keeps serving
    // further pf_launch_fs_kernel calls (timing), but stepping and read-out need pf_set_fields first.
    c->state = ST_TIMING;
    c->s2c_valid = true;
    return rc;
}
int pf_num_fs_kernels(const pf_ctx *c)
{
    if (!c) return 0;
    return c->p.ndim == 2 ? 2 : 4;
}
double pf_fs_kernel_ms(pf_ctx *c, int which) { return (c && which >= 0 && which < c->nk) ? c->kms[which] : -1.0; }
const char *pf_fs_kernel_name(const pf_ctx *c, int which)
{
    static const char *k2d[] = {"row_c2r_nonlinear_r2c", "col_y_fft_update_ifft"};
    static const char *k3d[] = {"row_c2r_nonlinear_r2c", "col_y_fwd", "col_z_fft_update_ifft", "col_y_inv"};
    if (!c || which < 0 || which >= pf_num_fs_kernels(c)) return "";
    return c->p.ndim == 2 ? k2d[which] : k3d[which];
}

}  // extern "C"
