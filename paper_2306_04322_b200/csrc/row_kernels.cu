// row_kernels.cu -- the x-direction kernel of the Fourier-spectral step.
//
// State between steps is the "z-form": for every grid row (fixed y, z) and field, the length-M = nx/2
// complex transform of the packed row  z[n] = u[2n] + i u[2n+1].  The Hermitian split that turns it
// into the true half spectrum is pointwise in y and lives in the column kernels, so this kernel is
// pure complex FFT work:
//
//   ROW_STEP:  load z-form of c, eta_1..p      -> inverse FFT_M -> real samples c, eta_i (registers)
//              -> share the samples of the F fields of the row through shared memory
//              -> g = df_chem/dc                                (Alg. 1; f_chem PAPER.md:46)
//                 w_i = eta_i - dt L df_chem/deta_i             (right-hand side of Eq. 13, PAPER.md:107,
//                                                                formed in real space: F is linear)
//              -> forward FFT_M -> store z-form of g (own array) and of w_i (over eta_i's state)
//   ROW_SET:   real fields -> forward FFT_M -> z-form state
//   ROW_GET:   z-form state -> inverse FFT_M / M -> real fields
//
// Thread layout: block = RB rows x F fields x TT = M/E threads; thread (r, f, j) owns elements
// j + q*TT of the transform of field f of row r (fft_core.cuh). One barrier-separated shared-memory
// exchange per FFT stage boundary plus one for the nonlinear coupling.
#include <type_traits>
#include "pf_kernels.cuh"

#ifndef PF_ROW_THREADS
#define PF_ROW_THREADS 256
#endif
#ifndef PF_ROW_E1024
#define PF_ROW_E1024 8
#endif
#ifndef PF_ROW_REGS_BIG
#define PF_ROW_REGS_BIG 80
#endif
#define PF_ROW_REGS(T, M, E) ((((E) >= 16) && sizeof(T) == 8) ? 128 : ((M) >= 256) ? PF_ROW_REGS_BIG : 64)
// fp64 rows of nx = 2048 with 7..9 fields: F * 128 threads at 80 registers do not fit an SM (register file, and 1152 >
// 1024 threads at F = 9), so these run 16 elements per thread: F * 64 <= 576 threads = 18 warps, i.e. up to 5 warps on one
// of the four 16 K-register sub-partitions -> at most 102 registers per thread
#define PF_ROW_REGS_WIDE 96
#ifndef PF_ROW_LOGPAD
#define PF_ROW_LOGPAD(C) (sizeof(C) == 8 ? 4 : 3)
#endif

namespace pf {

template <typename C, int LOGPAD> struct RowBuf {
    C *base;
    __device__ __forceinline__ void st(int i, C v) { base[i + (i >> LOGPAD)] = v; }
    __device__ __forceinline__ C ld(int i) const { return base[i + (i >> LOGPAD)]; }
    template <int N, int E, int NS> __device__ __forceinline__ void store(const C (&v)[E], int j) { exchange_store<N, E, NS>(v, j, *this); }
    template <int N, int E> __device__ __forceinline__ void load(C (&v)[E], int j) const { exchange_load<N, E>(v, j, *this); }
};
struct CtaSync { __device__ __forceinline__ void operator()() const { __syncthreads(); } };
// a transform carried by exactly one warp exchanges through its own buffer: warp-level synchronisation is enough,
// and the warps of an SM drift apart (their fp64 and shared-memory phases overlap instead of alternating)
struct WarpSync { __device__ __forceinline__ void operator()() const { __syncwarp(); } };
// a transform carried by several warps: named barrier over exactly its TT threads (ids 1..15; id 0 is __syncthreads),
// so the transforms of a CTA (fields, rows) drift apart between the points where the nonlinear terms couple them
struct GroupSync {
    int id, n;
    __device__ __forceinline__ void operator()() const { asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(n) : "memory"); }
};


template <int M, int E> __host__ __device__ constexpr int row_pitch() { return M + (M >> 3) + 1; }

// Register cap: the kernel is bound by fp64 issue and shared-memory exchange latency, so resident warps matter more
// than the last few registers (measured on B200: 94 -> 80 registers: 1024^2 row kernel 28.1 -> 26.4 us; 64 at
// nx = 256: 394 -> 317 us at 256^3).
// NF > 0: the field count as a compile-time constant (the loops over the fields of a point unroll); NF == 0: from p.F (ROW_SET / ROW_GET,
// which do not loop over fields)
template <typename T, int M, int E, int MODE, int REGS, int NF>
__global__ void __maxnreg__(REGS) row_kernel(const RowParams<T> p)
{
#ifdef PF_DBG_EMPTY
    return;
#endif
    typedef typename V2<T>::type C;
    constexpr int TT = M / E;
    constexpr int MP = row_pitch<M, E>();
    // one element of padding per 128-byte line of the exchange buffer: 8 fp64 / 16 fp32 complex values (with one per 8 the
    // first-stage scatter of the fp32 transforms ran at twice the minimum number of wavefronts, profiles/r2_ncu_full.md)
    constexpr int LP = PF_ROW_LOGPAD(C);
#ifdef PF_TRACE
    TraceScope trace(p.trace, 0);
#endif
    extern __shared__ __align__(16) unsigned char smem_raw[];
    C *smem = reinterpret_cast<C *>(smem_raw);

    const int F = NF ? NF : p.F;
    const int tid = threadIdx.x;
    const int j = tid & (TT - 1);
    // transform `tid / TT` of the CTA is field f of row r, FIELD-major: the two or more transforms that share a warp when TT < 32
    // then belong to the same field (RB is even there), so a warp never runs both the c branch and the eta branch of the
    // nonlinear section
    const int RB = blockDim.x / (TT * F);
    const int f = (tid / TT) / RB;
    const int r = (tid / TT) - f * RB;
    const int rf = r * F + f;                          // exchange buffer of this transform
    const long row = (long)blockIdx.x * RB + r;
    const bool valid = row < p.nrows;
    RowBuf<C, LP> buf{smem + (long)rf * MP};
    const CtaSync sync;
    const int rf_sync = threadIdx.x / TT;              // transform index within the CTA (at most 9 when TT > 32)

    grid_dependency_wait();
    grid_dependents_launch();

    C v[E];
    if (MODE == ROW_SET) {
        const C *src = reinterpret_cast<const C *>(p.real + f * p.rfs + row * (2L * M));
#pragma unroll
        for (int q = 0; q < E; ++q) v[q] = valid ? src[j + q * TT] : mk<T>(0, 0);
    } else {
        const C *src = p.zst + f * p.zfs + row * M;
#pragma unroll
        for (int q = 0; q < E; ++q) v[q] = valid ? cswap(src[j + q * TT]) : mk<T>(0, 0);   // swap: inverse via forward
        if constexpr (TT <= 32) fft_forward<M, E>(v, j, p.tw, buf, WarpSync());
        else fft_forward<M, E>(v, j, p.tw, buf, GroupSync{1 + rf_sync, TT});
        const T s = T(1) / T(M);
#pragma unroll
        for (int q = 0; q < E; ++q) v[q] = mk<T>(v[q].y * s, v[q].x * s);                    // swap back, normalise
    }

    if (MODE == ROW_GET) {
        C *dst = reinterpret_cast<C *>(p.real + f * p.rfs + row * (2L * M));
        if (valid) {
#pragma unroll
            for (int q = 0; q < E; ++q) dst[j + q * TT] = v[q];
        }
        return;
    }

    if (MODE == ROW_STEP) {
        // v[q] = (u_f[2n], u_f[2n+1]) at n = j + q*TT. Share across the fields of the row.
        sync();
#pragma unroll
        for (int q = 0; q < E; ++q) buf.st(j + q * TT, v[q]);
        sync();
        const C *rowbase = smem + (long)(r * F) * MP;
#pragma unroll
        for (int q = 0; q < E; ++q) {
            const int n = j + q * TT;
            const int np = n + (n >> LP);
            if (f == 0) {
                T h0 = 0, h1 = 0;                        // h(eta) = sum_i eta_i^3 (6 eta_i^2 - 15 eta_i + 10)
                for (int ff = 1; ff < F; ++ff) {
                    const C e = rowbase[(long)ff * MP + np];
                    h0 += h_term(e.x); h1 += h_term(e.y);
                }
                v[q] = mk<T>(dfdc(p.m, v[q].x, h0), dfdc(p.m, v[q].y, h1));
            } else {
                T s0 = 0, s1 = 0;                        // sum_j eta_j^2 (own field included)
                for (int ff = 1; ff < F; ++ff) {
                    const C e = rowbase[(long)ff * MP + np];
                    s0 += e.x * e.x; s1 += e.y * e.y;
                }
                const C c = rowbase[np];
                v[q] = mk<T>(v[q].x - p.m.dtL * dfdeta(p.m, c.x, v[q].x, s0),
                             v[q].y - p.m.dtL * dfdeta(p.m, c.y, v[q].y, s1));
            }
        }
    }

    // with warp-level exchange barriers the buffers the other fields' threads have just read need a CTA barrier
    if (MODE == ROW_STEP) sync();
    if constexpr (TT <= 32) fft_forward<M, E>(v, j, p.tw, buf, WarpSync());
    else fft_forward<M, E>(v, j, p.tw, buf, GroupSync{1 + rf_sync, TT});

    C *dst = (MODE == ROW_STEP && f == 0) ? (p.zg + row * M) : (p.zst + f * p.zfs + row * M);
    if (valid) {
#pragma unroll
        for (int q = 0; q < E; ++q) dst[j + q * TT] = v[q];
    }
#ifdef PF_TRACE
    if (MODE == ROW_STEP) trace.finish();
#endif
}

template <typename T, int M, int E, int MODE, int REGS, int NF = 0>
static cudaError_t launch_row_inst(const RowParams<T> &p, cudaStream_t s)
{
    typedef typename V2<T>::type C;
    constexpr int TT = M / E;
    const int per_row = TT * p.F;
    // the warps of a CTA are dealt round-robin to four sub-partitions of 16 K registers each
    if (per_row > 1024 || ((per_row / 32 + 3) / 4) * 32 * REGS > 16384) return cudaErrorInvalidConfiguration;
    int RB = PF_ROW_THREADS / per_row;
    if (RB > p.nrows / 296) RB = p.nrows / 296;      // small grids: at least two CTAs per SM before rows are batched
    if (RB < 1) RB = 1;
    if (RB > p.nrows) RB = p.nrows;
    if (TT < 32 && RB >= 32 / TT) RB -= RB % (32 / TT);          // whole warps per field (see the kernel)
    const int threads = RB * per_row;
    const size_t smem = (size_t)RB * p.F * row_pitch<M, E>() * sizeof(C);
    auto kern = row_kernel<T, M, E, MODE, REGS, NF>;
    if (smem > 48 * 1024) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
    }
    if (p.carveout > 0) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributePreferredSharedMemoryCarveout, p.carveout);
        if (e != cudaSuccess) return e;
    }
    const unsigned grid = (unsigned)((p.nrows + RB - 1) / RB);
    return launch_pdl(kern, dim3(grid), dim3(threads), smem, s, p.pdl != 0, p);
}

template <typename T, int M, int E, int REGS = PF_ROW_REGS(T, M, E)>
static cudaError_t launch_row_mode(int mode, const RowParams<T> &p, cudaStream_t s)
{
    switch (mode) {
    case ROW_SET:  return launch_row_inst<T, M, E, ROW_SET, REGS>(p, s);
    case ROW_STEP:
        switch (p.F) {                     // field count as a template parameter (see the kernel)
        case 1: return launch_row_inst<T, M, E, ROW_STEP, REGS, 1>(p, s);
        case 2: return launch_row_inst<T, M, E, ROW_STEP, REGS, 2>(p, s);
        case 3: return launch_row_inst<T, M, E, ROW_STEP, REGS, 3>(p, s);
        case 4: return launch_row_inst<T, M, E, ROW_STEP, REGS, 4>(p, s);
        case 5: return launch_row_inst<T, M, E, ROW_STEP, REGS, 5>(p, s);
        case 6: return launch_row_inst<T, M, E, ROW_STEP, REGS, 6>(p, s);
        case 7: return launch_row_inst<T, M, E, ROW_STEP, REGS, 7>(p, s);
        case 8: return launch_row_inst<T, M, E, ROW_STEP, REGS, 8>(p, s);
        case 9: return launch_row_inst<T, M, E, ROW_STEP, REGS, 9>(p, s);
        }
        return launch_row_inst<T, M, E, ROW_STEP, REGS>(p, s);
    case ROW_GET:  return launch_row_inst<T, M, E, ROW_GET, REGS>(p, s);
    }
    return cudaErrorInvalidValue;
}

template <typename T> cudaError_t launch_row(int mode, int nx, const RowParams<T> &p, cudaStream_t s)
{
    switch (nx / 2) {
    case 8:    return launch_row_mode<T, 8, 8>(mode, p, s);
    case 16:   return launch_row_mode<T, 16, 8>(mode, p, s);
    case 32:   return launch_row_mode<T, 32, 8>(mode, p, s);
    case 64:   return launch_row_mode<T, 64, 8>(mode, p, s);
    case 128:  return launch_row_mode<T, 128, 8>(mode, p, s);
    case 256:  return launch_row_mode<T, 256, 8>(mode, p, s);
    case 512:  return launch_row_mode<T, 512, 8>(mode, p, s);
    // fp32 at nx = 2048: 16 elements per thread (the bytes an fp64 thread holds with 8), two CTAs per SM
    case 1024:
        if constexpr (sizeof(T) == 4) return launch_row_mode<T, 1024, 16>(mode, p, s);
        else {
            if (p.F * (1024 / PF_ROW_E1024) * PF_ROW_REGS(T, 1024, PF_ROW_E1024) > 65536)      // F >= 7
                return launch_row_mode<T, 1024, 16, PF_ROW_REGS_WIDE>(mode, p, s);
            return launch_row_mode<T, 1024, PF_ROW_E1024>(mode, p, s);
        }
    }
    return cudaErrorInvalidValue;
}

template cudaError_t launch_row<double>(int, int, const RowParams<double> &, cudaStream_t);
template cudaError_t launch_row<float>(int, int, const RowParams<float> &, cudaStream_t);

}  // namespace pf
