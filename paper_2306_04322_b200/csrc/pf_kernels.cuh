// pf_kernels.cuh -- parameter blocks and launch entry points shared by the kernel translation units
// and the host library (pf.cu). Product code; nothing here is shared with oracle/.
#pragma once
#include <cuda_runtime.h>
#include "fft_core.cuh"

namespace pf {

// Model coefficients in the arithmetic type of the kernels (Eqs. 1-3, 12-15).
template <typename T> struct Model {
    T rho2, c_alpha, c_beta, w, alpha;     // f_chem
    T kappa_c, kappa_eta;
    T dt, M, L;
    T dtM, dtL;                            // dt*M, dt*L            (Eqs. 12-13)
    T dtMkc, dtLke;                        // dt*M*kappa_c, dt*L*kappa_eta   (Eqs. 14-15)
    // derived constants of the pointwise derivatives (dfdc, dfdeta below), formed once on the host in double
    T gA0, gA1, gA2;                       // df/dc = gA0 c - gA1 - gA2 h:  2 rho2, 2 rho2 c_alpha, 2 rho2 (c_beta - c_alpha)
    T eB0, eB1;                            // 30 (f^beta - f^alpha) = eB0 - eB1 c:  30 rho2 (c_beta^2 - c_alpha^2), 60 rho2 (c_beta - c_alpha)
    T eW2, eW4a;                           // 2 w, 4 alpha w
    int n_eta;
};

// -DPF_TRACE builds (profiles/: CTA timelines): every CTA of the step kernels appends {kind, %smid, start, end} (%globaltimer,
// ns) to a buffer the context dumps at pf_destroy into the file named by PF_TRACE_FILE. Never part of the default library.
struct TraceBuf { unsigned long long n, cap; unsigned long long rec[1]; };
#if defined(PF_TRACE) && defined(__CUDACC__)
#define PF_TRACE_FIELD TraceBuf *trace;
struct TraceScope {
    TraceBuf *b; unsigned long long t0; int kind;
    __device__ __forceinline__ TraceScope(TraceBuf *buf, int k) : b(buf), kind(k)
    {
        asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t0));
    }
    __device__ __forceinline__ void finish()
    {
        __syncthreads();
        if (b && threadIdx.x == 0) {
            unsigned long long t1; unsigned sm;
            asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t1));
            asm volatile("mov.u32 %0, %%smid;" : "=r"(sm));
            const unsigned long long i = atomicAdd(&b->n, 1ull);
            if (i < b->cap) { b->rec[3 * i] = ((unsigned long long)kind << 32) | sm; b->rec[3 * i + 1] = t0; b->rec[3 * i + 2] = t1; }
        }
    }
};
#elif defined(PF_TRACE)
#define PF_TRACE_FIELD TraceBuf *trace;
#else
#define PF_TRACE_FIELD
#endif

enum RowMode { ROW_SET = 0, ROW_STEP = 1, ROW_GET = 2 };

// x-direction kernel. "z-form" of a real row u[0..nx): Z = FFT_{nx/2}( u[2n] + i u[2n+1] ), nx/2 complex values.
template <typename T> struct RowParams {
    typedef typename V2<T>::type C;
    C       *zst;            // [F][nrows][M]   state, z-form (M = nx/2)
    C       *zg;             // [nrows][M]      z-form of g = df_chem/dc (ROW_STEP output)
    T       *real;           // [F][nrows][nx]  real fields (ROW_SET input / ROW_GET output)
    const C *tw;             // exp(-2 pi i k / M), k < M
    long     zfs;            // field stride of zst in complex elements (= nrows*M)
    long     rfs;            // field stride of real in reals (= nrows*nx)
    int      nrows;          // ny*nz
    int      F;              // 1 + n_eta
    int      pdl;            // launch with programmatic stream serialization
    int      carveout;       // preferred shared-memory carve-out in percent (0: the driver's choice), see col2d_shape()
    Model<T> m;
    PF_TRACE_FIELD
};

// Column-kernel modes (see col_kernels.cu)
enum ColMode {
    COL_2D_LAST   = 0,   // z-form pairs -> unpack, FFT_y, spectral update, IFFT_y, repack -> z-form
    COL_3D_MIDFWD = 1,   // z-form pairs -> unpack, FFT_y -> half-spectrum planes [nz][ny][P2]
    COL_3D_MIDINV = 2,   // half-spectrum planes -> IFFT_y, repack -> z-form
    COL_3D_LAST   = 3,   // half-spectrum columns along z: FFT_z, spectral update, IFFT_z (in place)
    COL_2D_ENERGY = 4,   // z-form pairs -> unpack, FFT_y, accumulate sum w_k |xi|^2 |u^|^2
    COL_3D_ENERGY = 5    // half-spectrum columns along z: FFT_z, accumulate
};

template <typename T> struct ColParams {
    typedef typename V2<T>::type C;
    const C *in0;            // input of slot s: in0 + s*in_fs  (eta fields: w = eta - dt L h; slot 0: the c state)
    const C *in1;            // update modes with has_c: g = df/dc (same layout as slot 0 of in0)
    C       *out;            // output of slot s: out + s*out_fs
    C       *park;           // update modes with has_c: scratch for dt M |xi|^2 g^, one complex per spectral mode (+ padding)
    const C *alt_in;         // if non-null, slot 0 reads alt_in and writes alt_out instead (3D y-forward of g)
    C       *alt_out;
    int      has_c;          // update modes: slot 0 is the Cahn-Hilliard field (needs in1). 1: c^ re-transformed, dt M |xi|^2 g^ parked;
                             // 2: c^ carried in `park`; 3: one-off pass that fills the carried spectrum from in0 (slot 0 only)
    int      pdl;            // launch with programmatic stream serialization
    long     in_fs, out_fs;  // slot strides (blockIdx.z)
    long     in_bs, out_bs;           // batch strides (blockIdx.y; 3D mid kernels: z planes)
    long     in_rs, out_rs;           // stride between consecutive elements along the FFT axis
    int      M;              // nx/2
    int      P2;             // pitch of half-spectrum planes (>= M+1, multiple of 8)
    int      ncols;          // plain-column modes: number of columns (3D last: ny*P2)
    const C *tw;             // exp(-2 pi i k / N), N = length of the FFT axis
    const C *twx;            // exp(-2 pi i k / nx), k <= M/2   (Hermitian pack/unpack)
    const T *kx2;            // |xi_x|^2 per kx, P2 entries (zero padded)
    const T *ky2;            // per ky (2D last: the FFT axis; 3D last: the middle axis)
    const T *kz2;            // per kz (3D last: the FFT axis)
    double  *acc;            // energy modes: accumulator (one double per field)
    int     *queue;          // persistent kernels (wcol_kernels.cu): {next item, CTAs finished}, zero between launches
    Model<T> m;
    PF_TRACE_FIELD
};

// 2D last-axis kernel with carried c^ and a static balanced schedule (col2d_kernels.cu)
enum Col2dOp {
    COL2D_ETA    = 0,   // Allen-Cahn block: unpack, FFT_y, Eq. 15, IFFT_y, repack                       (two rounds)
    COL2D_C_FWD  = 1,   // Cahn-Hilliard block, first half: unpack g, FFT_y, Eq. 14 on the carried c^    (one round)
    COL2D_C_INV  = 2,   // second half: carried c^ -> IFFT_y, repack                                     (one round)
    COL2D_C_FULL = 3,   // both halves in one CTA, values kept in registers
    COL2D_C_INIT = 4    // z-form of c -> unpack, FFT_y -> carry (after pf_set_fields / FD steps)
};
template <typename T> struct Col2dParams {
    typedef typename V2<T>::type C;
    C       *zst;            // [F][B][ny][M] z-form state of B replicas; slot s at zst + s*zfs (slot 0 = c, written by C_INV / C_FULL)
    const C *zg;             // [B][ny][M] z-form of g = df/dc
    C       *carry;          // c^ in the kernel's thread-linear order: [B*nblk][E][THREADS]
    long     zfs;
    int      M;              // nx/2 = pitch of the z-form rows
    int      nblk;           // column blocks per replica (items carry replica * nblk + block)
    int      per_cta;        // items per CTA in sched (padded with -1; at most Col2dShapeInfo::max_items)
    const int *sched;        // [grid][per_cta] items: op | slot << 4 | block << 8
    int     *flags;          // [B*nblk] C_FWD -> C_INV hand-off, zero between launches
    unsigned *ticket;        // place counter (zero between launches; wraps with the last CTA); nullptr: place = blockIdx.x
    int      pdl;
    const C *tw;             // exp(-2 pi i k / ny)
    const C *twx;            // exp(-2 pi i k / nx), k <= M/2
    const T *kx2, *ky2;      // |xi_x|^2 per kx (M+1 entries), |xi_y|^2 per ky
    Model<T> m;
    PF_TRACE_FIELD
};
// carveout_pct: the shared-memory carve-out (percent of the SM's maximum) the kernel runs with. An SM switches carve-out
// only when it is idle, so a kernel launched with programmatic stream serialization becomes resident under its
// predecessor's last CTAs only if both run with the SAME carve-out: the x kernel is given this value too.
struct Col2dShapeInfo { int tp, e, threads, max_items, nblk, slots, carveout_pct; long carry_elems; };

// small 2D grids resident in the shared memory of a thread-block cluster (sgrid_kernels.cu)
template <typename T> struct SgParams {
    typedef typename V2<T>::type C;
    C       *zst;            // [F][B][ny][M] z-form state in global memory: read at the start, written at the end
    long     zfs;            // field stride (= B*ny*M)
    int      F;              // 1 + n_eta
    int      nsteps;         // steps of Algorithm 1 to run inside the launch
    const C *tw_m, *tw_y;    // exp(-2 pi i k / M), exp(-2 pi i k / ny)
    const C *twx;            // exp(-2 pi i k / nx), k <= M/2
    const T *kx2, *ky2;      // |xi_x|^2 (M+1 entries), |xi_y|^2
    Model<T> m;
};

// FD path
template <typename T> struct FdParams {
    const T *c, *eta;        // time-t fields
    T       *c_new, *eta_new;
    int      nx, ny, nz;
    long     N;              // nx*ny*nz
    long     fs;             // stride between the eta fields (N x replicas of a batched 2D context; replica b at + b*N)
    int      nbatch;         // replicas (2D only: blockIdx.z)
    T        rdx2[3];        // 1/dx^2 per axis (rdx2[2] = 0 in 2D)
    Model<T> m;
};

template <typename T> struct EnergyParams {
    const T *c, *eta;
    int      nx, ny, nz;
    long     N;
    T        rdx[3];         // 1/dx per axis (0 in z for 2D)
    int      gradient_kind;  // 1: add forward-difference gradient terms; 0: chemical part only
    double  *acc;            // [2 + n_eta]: chem, grad c, grad eta_i
    Model<T> m;
};

// ---- launchers (defined in the .cu files; return cudaGetLastError()) ----
template <typename T> cudaError_t launch_row(int mode, int nx, const RowParams<T> &p, cudaStream_t s);
template <typename T> cudaError_t launch_col(int mode, int nfft, int nslots, int nbatch, const ColParams<T> &p, cudaStream_t s);
// persistent pipelined form of COL_2D_LAST for long fp64 axes; cudaErrorNotSupported when the shape has none
template <typename T> cudaError_t launch_wcol2d(int nfft, int nslots, const ColParams<T> &p, cudaStream_t s);
template <typename T> cudaError_t col2d_shape(int nfft, int M, Col2dShapeInfo *o);
template <typename T> cudaError_t launch_col2d(int nfft, const Col2dParams<T> &p, int grid, cudaStream_t s);
template <typename T> int sgrid_plan(int nx, int ny, int F, int want);
template <typename T> cudaError_t launch_sgrid(int nx, int ny, const SgParams<T> &p, int cs, int nbatch, cudaStream_t s);
template <typename T> cudaError_t launch_fd_fused2d(const FdParams<T> &p, cudaStream_t s);
// 2D, nx >= 64, ny >= 16: pair-wide tile kernel (fd2d_kernels.cu); cudaErrorNotSupported otherwise
template <typename T> cudaError_t launch_fd2d_pair(const FdParams<T> &p, cudaStream_t s);
template <typename T> cudaError_t launch_fd_fused3d(const FdParams<T> &p, cudaStream_t s);
// 3D, nx >= 64, at most four order parameters (fd3d_kernels.cu); cudaErrorNotSupported otherwise
template <typename T> cudaError_t launch_fd3d_march(const FdParams<T> &p, cudaStream_t s);
template <typename T> cudaError_t launch_energy(const EnergyParams<T> &p, cudaStream_t s);

#if defined(__CUDACC__)
// Programmatic dependent launch: a kernel launched with the attribute may start while its predecessor in the
// stream is still running; it must not touch data the predecessor produces (or still reads) before
// grid_dependency_wait(), which returns once the predecessor grid has completed and flushed.
__device__ __forceinline__ void grid_dependency_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void grid_dependents_launch() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

template <typename K, typename... P>
static inline cudaError_t launch_pdl(K kern, dim3 grid, dim3 block, size_t smem, cudaStream_t s, bool pdl, const P &...params)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = s;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at; cfg.numAttrs = pdl ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, kern, params...);
}
#endif

// pointwise model, shared by the row kernel, the FD kernels and the energy kernel --------------------
// h(eta) = sum eta^3 (6 eta^2 - 15 eta + 10); g(eta) = sum eta^2 (1-eta)^2 + alpha sum_i sum_{j!=i} eta_i^2 eta_j^2
// f_chem = rho2 (c-c_alpha)^2 (1-h) + rho2 (c_beta-c)^2 h + w g
template <typename T> PF_HD T h_term(T e) { return e * e * e * (e * (T(6) * e - T(15)) + T(10)); }
// d f_chem / dc = 2 rho2 [ (c - c_alpha)(1 - h) - (c_beta - c) h ] = 2 rho2 (c - c_alpha) - 2 rho2 (c_beta - c_alpha) h
template <typename T> PF_HD T dfdc(const Model<T> &m, T c, T h)
{
    return (m.gA0 * c - m.gA1) - m.gA2 * h;
}
// d f_chem / d eta_i = (f^beta - f^alpha) 30 eta^2 (1-eta)^2 + w [ 2 eta (1-eta)(1-2 eta) + 4 alpha eta (s2 - eta^2) ],
// s2 = sum_j eta_j^2 (each unordered pair appears twice in the ordered double sum of g -> 4 alpha);
// f^beta - f^alpha = rho2 [(c_beta - c)^2 - (c - c_alpha)^2] = rho2 (c_beta - c_alpha)(c_beta + c_alpha - 2 c) is linear in c
template <typename T> PF_HD T dfdeta(const Model<T> &m, T c, T e, T s2)
{
    const T fba30 = m.eB0 - m.eB1 * c;             // 30 (f^beta - f^alpha)
    const T u = e - e * e;                         // eta (1 - eta)
    const T b = u * (T(1) - T(2) * e);
    const T d = e * (s2 - e * e);
    return fba30 * (u * u) + m.eW2 * b + m.eW4a * d;
}

}  // namespace pf
