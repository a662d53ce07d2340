// col_kernels.cu -- strided-direction kernels of the Fourier-spectral step.
//
// A CTA owns SLOTS = 2*TP adjacent columns and all N elements of each along the FFT axis. Thread (slot, j) holds
// elements j + q*TT (q < E, TT = N/E) of ONE column in registers (fft_core.cuh), before and after every transform,
// so the pointwise work is register local. The slot is the fastest thread index: consecutive lanes own consecutive
// columns, every global access of a warp is made of contiguous 16*SLOTS-byte (fp64) pieces, and the strided
// "transpose" happens in registers plus one shared-memory exchange per FFT stage boundary (col_buf.cuh). One column
// per thread keeps the kernel at 64 registers and N*SLOTS*16 bytes of shared memory per CTA (64 KB at N = 1024), so
// two to four CTAs share an SM, start and finish at different times, and one CTA's loads and stores overlap the
// transforms of the others.
//
// In the pair modes the columns of a CTA are TP mirror pairs (u, M-u) of the z-form (row_kernels.cu): with
//   E = (Z_u + conj Z_{M-u})/2,  O = -(i/2)(Z_u - conj Z_{M-u}),  W = exp(-2 pi i u / nx)
// the true half-spectrum columns are  U_u = E + W O  (side 0) and  U_{M-u} = conj(E - W O)  (side 1), pointwise
// along the column; u = 0 yields the DC and Nyquist columns from Z_0 alone and u = M/2 is its own mirror. Both
// threads of a pair read both z columns (the second read hits L1); after the inverse transform they exchange
// their results with one warp shuffle and each writes its own z column. The spectral update itself is
//   c^   <- ( c^ - dt M |xi|^2 g^ ) / ( 1 + dt M kappa_c |xi|^4 )        Eqs. 12, 14
//   eta^ <- w^ / ( 1 + dt L kappa_eta |xi|^2 ),  w = eta - dt L h        Eqs. 13, 15
// with |xi|^2 = kx2 + ky2 (+ kz2) from 1-D tables (Eq. 16/19 or the FS-FD variants).
//
// Field slots (blockIdx.z): in the update modes slot 0 is c, which needs two forward transforms on the same columns:
// its CTAs first transform g = df/dc, scale it by dt M |xi|^2 and park it in global memory (each thread reads back
// what it wrote itself; the 8 MB stay in L2), then transform c^, combine, invert and store.
#include "pf_kernels.cuh"
#include "col_buf.cuh"
#include "wfft.cuh"

// -DPF_WFFT: long fp64 axes use the warp-tile transform of wfft.cuh (one shared-memory exchange per transform, the rest
// in warp shuffles) instead of the Stockham path of fft_core.cuh. Measured on B200 and NOT the default: it removes 23 % of
// the shared-memory wavefronts and two thirds of the barriers but adds 31 % instructions (the selects of the shuffle
// transposes) and comes out level at 1024^2 and slower at 512^2 / 2048^2 (profiles/r2_col_variants.md)
#ifndef PF_WFFT_MIN_N
#define PF_WFFT_MIN_N 512
#endif

// column pairs per CTA at the longer axes (tuned on B200)
#ifndef PF_COL_THREADS_PER_SM
#define PF_COL_THREADS_PER_SM 1024
#endif
#ifndef PF_TP_32
#define PF_TP_32 8
#endif
#ifndef PF_TP_64
#define PF_TP_64 4
#endif
#ifndef PF_TP_128
#define PF_TP_128 4
#endif
#ifndef PF_TP_256
#define PF_TP_256 4
#endif
#ifndef PF_TP_512
#define PF_TP_512 2
#endif
#ifndef PF_F32_TP_1024
#define PF_F32_TP_1024 4
#endif
#ifndef PF_F32_TP_2048
#define PF_F32_TP_2048 2
#endif
#ifndef PF_TP_1024
#define PF_TP_1024 2
#endif
#ifndef PF_TP_2048
#define PF_TP_2048 2
#endif

namespace pf {

__device__ __forceinline__ double rcp(double x) { return __drcp_rn(x); }
__device__ __forceinline__ float rcp(float x) { return __frcp_rn(x); }

__device__ __forceinline__ double2 shfl_xor1(double2 v)
{
    return make_double2(__shfl_xor_sync(0xffffffffu, v.x, 1), __shfl_xor_sync(0xffffffffu, v.y, 1));
}
__device__ __forceinline__ float2 shfl_xor1(float2 v)
{
    return make_float2(__shfl_xor_sync(0xffffffffu, v.x, 1), __shfl_xor_sync(0xffffffffu, v.y, 1));
}

struct CtaSync { __device__ __forceinline__ void operator()() const { __syncthreads(); } };

template <int N, int E, int TP> struct ColShape {
    static constexpr int TT = N / E;
    static constexpr int SLOTS = 2 * TP;
    static constexpr int THREADS = SLOTS * TT;                           // whole warps
    static constexpr int BUDGET = PF_COL_THREADS_PER_SM;                 // resident threads per SM the register cap is set for (1024: 64 registers)
    static constexpr int MINB = (THREADS >= BUDGET) ? 1 : ((BUDGET / THREADS > 32) ? 32 : BUDGET / THREADS);
    static constexpr int LR = (E >= 16) ? 4 : 3;                         // log2 of the first-stage radix
#ifdef PF_WFFT
    static constexpr bool WF = (E == 8 && TP == 2 && N >= PF_WFFT_MIN_N && N >= 256 && N <= 2048);
#else
    static constexpr bool WF = false;
#endif
};

template <typename T, int N, int E, int TP, int MODE>
__global__ void __launch_bounds__(ColShape<N, E, TP>::THREADS, ColShape<N, E, TP>::MINB)
col_kernel(const ColParams<T> p)
{
#ifdef PF_DBG_EMPTY
    return;
#endif
    typedef typename V2<T>::type C;
    typedef ColShape<N, E, TP> Sh;
    constexpr int TT = Sh::TT, SLOTS = Sh::SLOTS, GT = Sh::THREADS;
    constexpr bool PAIRS = (MODE == COL_2D_LAST || MODE == COL_3D_MIDFWD || MODE == COL_3D_MIDINV || MODE == COL_2D_ENERGY);
    constexpr bool PAIR_IN = (MODE == COL_2D_LAST || MODE == COL_3D_MIDFWD || MODE == COL_2D_ENERGY);
    constexpr bool PAIR_OUT = (MODE == COL_2D_LAST || MODE == COL_3D_MIDINV);
    constexpr bool ENERGY = (MODE == COL_2D_ENERGY || MODE == COL_3D_ENERGY);
    constexpr bool DO_FWD = (MODE != COL_3D_MIDINV);
    constexpr bool DO_UPD = (MODE == COL_2D_LAST || MODE == COL_3D_LAST);
    constexpr bool DO_INV = (MODE == COL_2D_LAST || MODE == COL_3D_LAST || MODE == COL_3D_MIDINV);
    constexpr bool LAST3D = (MODE == COL_3D_LAST || MODE == COL_3D_ENERGY);
    static_assert(GT % 32 == 0, "a CTA must be whole warps");

#ifdef PF_TRACE
    TraceScope trace(p.trace, 1 + MODE);
#endif
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int tid = threadIdx.x;
    const int sl = tid % SLOTS;                        // column slot: side = sl & 1, pair t = sl >> 1
    const int side = sl & 1;
    const int j = tid / SLOTS;
    const int M = p.M;
    const int slot = blockIdx.z;                       // field slot
    const long bz = blockIdx.y;
    const int ub = blockIdx.x;                         // block of SLOTS columns
    const bool c_cta = DO_UPD && p.has_c && slot == 0;

    constexpr bool WF = Sh::WF && sizeof(T) == 8;
    ColBuf<C, SLOTS, Sh::LR> buf{reinterpret_cast<C *>(smem_raw), sl};
    const CtaSync sync;
    // warp-tile kernels keep the twiddle table and the |xi|^2 table of the FFT axis in shared memory behind the exchange
    // buffer: every transform needs two twiddles and every update eight frequencies per thread, all of them scattered
    // 8/16-byte reads that miss L1 (ncu: 42 % of the load requests and as many L2 sectors as the field data)
    C *s_tw = reinterpret_cast<C *>(smem_raw) + (size_t)N * SLOTS;
    T *s_k2 = reinterpret_cast<T *>(s_tw + N);
#ifdef PF_NO_SMEM_TABLES
    constexpr bool TS = false;
#else
    constexpr bool TS = WF;
#endif
    WFft<T, WF ? N : 1024, TS> wf(reinterpret_cast<C *>(smem_raw), TS ? s_tw : p.tw, tid);
    // memory row and (after a forward transform) frequency index of register q
    auto rowq = [&](int q) -> int { if constexpr (WF) return wf.row(q); else return j + q * TT; };
    auto kq = [&](int q) -> int { if constexpr (WF) return wf.kidx(q); else return j + q * TT; };
    auto forward = [&](C (&x)[E]) { if constexpr (WF) wf.dif(x); else fft_forward<N, E>(x, j, p.tw, buf, sync); };
    auto transposed = [&](C (&x)[E]) { if constexpr (WF) wf.dit(x); else fft_forward<N, E>(x, j, p.tw, buf, sync); };

    // ---- which column ----
    bool valid = true;
    bool store_ok;                        // this thread writes its column
    int zcolA = 0, zcolB = 0;             // z-form columns of the pair (pitch M)
    int pcol = 0;                         // column index in plain arrays (half-spectrum planes)
    int kx;                               // kx of this thread's true spectral column
    T base2;                              // |xi|^2 contributions that are constant along the column
    C wx = mk<T>(1, 0);                   // exp(-2 pi i u / nx)
    if (PAIRS) {
        int u = ub * TP + (sl >> 1);
        valid = (u <= M / 2);
        if (!valid) u = 0;
        zcolA = u; zcolB = (M - u) & (M - 1);
        kx = side ? M - u : u;
        pcol = kx;
        store_ok = valid && (side == 0 || (PAIR_OUT ? zcolB != zcolA : kx != u));
        wx = p.twx[u];
        base2 = p.kx2[kx];
    } else {
        pcol = ub * SLOTS + sl;
        store_ok = true;
        kx = pcol % p.P2;
        base2 = p.kx2[kx] + p.ky2[pcol / p.P2];
    }

    // ---- arrays of this CTA ----
    const C *in;
    C *out;
    if (c_cta) {
        in = p.in1;                        // first pass: g = df/dc
        out = p.out;
    } else if (slot == 0 && p.alt_in) {
        in = p.alt_in; out = p.alt_out;
    } else {
        in = p.in0 + slot * p.in_fs;
        out = p.out + slot * p.out_fs;
    }
    in += bz * p.in_bs;
    out += bz * p.out_bs;

    C v[E];
    auto unpack = [&](C za, C zb) -> C {
        // E = (za + conj zb)/2, O = -(i/2)(za - conj zb)
        const C e = mk<T>(T(0.5) * (za.x + zb.x), T(0.5) * (za.y - zb.y));
        const C o = mk<T>(T(0.5) * (za.y + zb.y), T(-0.5) * (za.x - zb.x));
        const C wo = cmul(wx, o);
        return side ? cconj(csub(e, wo)) : cadd(e, wo);
    };
    auto load_columns = [&](const C *src) {
#ifdef PF_COL_OWNLOAD
        constexpr bool OWN = WF;                 // A/B build (profiles/r2_col_variants.md): measured slower
#else
        constexpr bool OWN = false;
#endif
        if constexpr (PAIR_IN && OWN) {
            // every thread loads ITS z column straight into v (eight independent 16-byte requests in flight, no landing
            // registers) and takes the mirror column from the neighbouring lane
            const C *mine = src + (side ? zcolB : zcolA);
#pragma unroll
            for (int q = 0; q < E; ++q) v[q] = mine[(long)rowq(q) * p.in_rs];
#pragma unroll
            for (int q = 0; q < E; ++q) {
                const C pv = shfl_xor1(v[q]);
                v[q] = side ? unpack(pv, v[q]) : unpack(v[q], pv);
            }
        } else if (PAIR_IN) {
#pragma unroll
            for (int q = 0; q < E; ++q) {
                const long i = rowq(q);
                v[q] = unpack(src[i * p.in_rs + zcolA], src[i * p.in_rs + zcolB]);
            }
        } else {
#pragma unroll
            for (int q = 0; q < E; ++q) v[q] = src[(long)rowq(q) * p.in_rs + pcol];
        }
    };

    const T *klast = LAST3D ? p.kz2 : p.ky2;
    if constexpr (TS) {
        for (int i = tid; i < N; i += GT) { s_tw[i] = p.tw[i]; s_k2[i] = klast[i]; }
        klast = s_k2;
        __syncthreads();
    }
    grid_dependency_wait();                // everything above touches constant tables only
    grid_dependents_launch();

    C *park = nullptr;
    bool carried = false;
    if (c_cta) {
        // thread-linear scratch of this CTA's columns: written and read back by the same thread
        park = p.park + ((bz * gridDim.x + ub) * (long)E) * GT + tid;
        if (p.has_c == 3) {
            // one-off (after pf_set_fields / FD steps): the carried spectrum c^ = FFT of the columns of c
            load_columns(p.in0 + bz * p.in_bs);
            forward(v);
#pragma unroll
            for (int q = 0; q < E; ++q) park[(long)q * GT] = v[q];
            return;
        }
        load_columns(in);
        forward(v);
        if (p.has_c == 2) {
            // c^ is CARRIED in the scratch array, as Algorithm 1 carries it: the Cahn-Hilliard columns cost
            // two transforms (g^, inverse) instead of three and nothing is parked
            //   c^ <- (c^ - dt M |xi|^2 g^) / (1 + dt M kappa_c |xi|^4)                           Eqs. 12, 14
            const T s = T(1) / T(N);
#pragma unroll
            for (int q = 0; q < E; ++q) {
                const T k2 = base2 + klast[kq(q)];
                const T d = rcp(T(1) + p.m.dtMkc * k2 * k2);
                const T a = p.m.dtM * k2;
                const C cq = park[(long)q * GT];
                const C cn = mk<T>((cq.x - a * v[q].x) * d, (cq.y - a * v[q].y) * d);
                park[(long)q * GT] = cn;
                v[q] = cscale(cn, s);
            }
            carried = true;
        } else {
            // Cahn-Hilliard with two forward transforms on the same columns: dt M |xi|^2 g^ is formed first and parked in
            // global memory (L2 resident), then c^ follows (2D legacy kernel, PF_COL3D_PARK=1)
#pragma unroll
            for (int q = 0; q < E; ++q) park[(long)q * GT] = cscale(v[q], p.m.dtM * (base2 + klast[kq(q)]));
            in = p.in0 + bz * p.in_bs;
        }
    }

    if (!carried) {
        load_columns(in);
        if (DO_FWD) forward(v);
    }

#ifndef PF_DBG_SKIP_UPDATE
    if (DO_UPD && !carried) {
        const T s = T(1) / T(N);
        if (c_cta) {
#pragma unroll
            for (int q = 0; q < E; ++q) {
                const T k2 = base2 + klast[kq(q)];
                const T d = s * rcp(T(1) + p.m.dtMkc * k2 * k2);
                const C gq = park[(long)q * GT];
                v[q] = mk<T>((v[q].x - gq.x) * d, (v[q].y - gq.y) * d);
            }
        } else {
#pragma unroll
            for (int q = 0; q < E; ++q) {
                const T k2 = base2 + klast[kq(q)];
                v[q] = cscale(v[q], s * rcp(T(1) + p.m.dtLke * k2));
            }
        }
    }
#endif

    if (ENERGY) {
        // sum over the full spectrum of |xi|^2 |u^|^2: columns with 0 < kx < M stand for their mirror too
        double acc = 0.0;
        const double wgt = (kx == 0 || kx == M) ? 1.0 : 2.0;
        if (store_ok && kx <= M) {
#pragma unroll
            for (int q = 0; q < E; ++q)
                acc += wgt * (double)(base2 + klast[kq(q)]) * ((double)v[q].x * v[q].x + (double)v[q].y * v[q].y);
        }
        double *red = reinterpret_cast<double *>(smem_raw);      // off the hot path: plain serial reduction
        __syncthreads();
        red[tid] = acc;
        __syncthreads();
        if (tid == 0) {
            double tot = 0.0;
            for (int w = 0; w < GT; ++w) tot += red[w];
            atomicAdd(p.acc + slot, tot);
        }
        return;
    }

    if (DO_INV) {
        // inverse = swap re/im, forward, swap re/im (unnormalised; the update folds 1/N in)
#pragma unroll
        for (int q = 0; q < E; ++q) v[q] = cswap(v[q]);
        transposed(v);
        const T s = DO_UPD ? T(1) : T(1) / T(N);
#pragma unroll
        for (int q = 0; q < E; ++q) v[q] = mk<T>(v[q].y * s, v[q].x * s);
    }

    if (PAIR_OUT) {
        // E = (Ua + conj Ub)/2, W O = (Ua - conj Ub)/2, Z_a = E + i O, Z_b = conj(E - i O); the partner (other side
        // of the pair) is the neighbouring lane
        const C wxc = cconj(wx);
        C *dst = out + (side ? zcolB : zcolA);
#pragma unroll
        for (int q = 0; q < E; ++q) {
            const C pv = shfl_xor1(v[q]);
            const C ua = side ? pv : v[q], ubv = side ? v[q] : pv;
            const C e = mk<T>(T(0.5) * (ua.x + ubv.x), T(0.5) * (ua.y - ubv.y));
            const C wo = mk<T>(T(0.5) * (ua.x - ubv.x), T(0.5) * (ua.y + ubv.y));
            const C io = cmul_pi(cmul(wxc, wo));
            const C z = side ? cconj(csub(e, io)) : cadd(e, io);
            if (store_ok) dst[(long)rowq(q) * p.out_rs] = z;
        }
    } else {
#pragma unroll
        for (int q = 0; q < E; ++q)
            if (store_ok) out[(long)rowq(q) * p.out_rs + pcol] = v[q];
    }
#ifdef PF_TRACE
    trace.finish();
#endif
}

template <typename T, int N, int E, int TP, int MODE>
static cudaError_t launch_col_inst(int nslots, int nbatch, const ColParams<T> &p, cudaStream_t s)
{
    typedef typename V2<T>::type C;
    typedef ColShape<N, E, TP> Sh;
    constexpr bool PAIRS = (MODE == COL_2D_LAST || MODE == COL_3D_MIDFWD || MODE == COL_3D_MIDINV || MODE == COL_2D_ENERGY);
    const int gx = PAIRS ? (p.M / 2 + TP) / TP : p.ncols / Sh::SLOTS;    // blocks of SLOTS columns
    size_t smem = (size_t)N * Sh::SLOTS * sizeof(C);
    if (Sh::WF && sizeof(T) == 8) smem += (size_t)N * (sizeof(C) + sizeof(T));                      // twiddle and |xi|^2 tables
    if (smem < (size_t)Sh::THREADS * sizeof(double)) smem = (size_t)Sh::THREADS * sizeof(double);   // energy reduction
    auto kern = col_kernel<T, N, E, TP, MODE>;
    if (smem > 48 * 1024) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
    }
    return launch_pdl(kern, dim3((unsigned)gx, (unsigned)nbatch, (unsigned)nslots), dim3(Sh::THREADS), smem, s, p.pdl != 0, p);
}

template <typename T, int N, int E, int TP>
static cudaError_t launch_col_mode(int mode, int nslots, int nbatch, const ColParams<T> &p, cudaStream_t s)
{
    switch (mode) {
    case COL_2D_LAST:   return launch_col_inst<T, N, E, TP, COL_2D_LAST>(nslots, nbatch, p, s);
    case COL_3D_MIDFWD: return launch_col_inst<T, N, E, TP, COL_3D_MIDFWD>(nslots, nbatch, p, s);
    case COL_3D_MIDINV: return launch_col_inst<T, N, E, TP, COL_3D_MIDINV>(nslots, nbatch, p, s);
    case COL_3D_LAST:   return launch_col_inst<T, N, E, TP, COL_3D_LAST>(nslots, nbatch, p, s);
    case COL_2D_ENERGY: return launch_col_inst<T, N, E, TP, COL_2D_ENERGY>(nslots, nbatch, p, s);
    case COL_3D_ENERGY: return launch_col_inst<T, N, E, TP, COL_3D_ENERGY>(nslots, nbatch, p, s);
    }
    return cudaErrorInvalidValue;
}

// nfft = length of the FFT axis. TP (column pairs per group) keeps a group at whole warps for short axes and the
// two exchange buffers of a CTA within 128 KB for long ones.
template <typename T> cudaError_t launch_col(int mode, int nfft, int nslots, int nbatch, const ColParams<T> &p, cudaStream_t s)
{
    // fp32: 16 elements per thread (the bytes an fp64 thread holds with 8) and twice the column pairs per CTA (32-byte pieces)
    if (sizeof(T) == 4) {
        switch (nfft) {
        case 1024: return launch_col_mode<T, 1024, 16, PF_F32_TP_1024>(mode, nslots, nbatch, p, s);
        case 2048: return launch_col_mode<T, 2048, 16, PF_F32_TP_2048>(mode, nslots, nbatch, p, s);
        }
    }
    switch (nfft) {
#ifndef PF_ONLY_N
    case 16:   return launch_col_mode<T, 16, 8, 8>(mode, nslots, nbatch, p, s);
    case 32:   return launch_col_mode<T, 32, 8, PF_TP_32>(mode, nslots, nbatch, p, s);
    case 64:   return launch_col_mode<T, 64, 8, PF_TP_64>(mode, nslots, nbatch, p, s);
    case 128:  return launch_col_mode<T, 128, 8, PF_TP_128>(mode, nslots, nbatch, p, s);
    case 256:  return launch_col_mode<T, 256, 8, PF_TP_256>(mode, nslots, nbatch, p, s);
    case 512:  return launch_col_mode<T, 512, 8, PF_TP_512>(mode, nslots, nbatch, p, s);
#endif
#if !defined(PF_ONLY_N) || PF_ONLY_N == 1024
    case 1024: return launch_col_mode<T, 1024, 8, PF_TP_1024>(mode, nslots, nbatch, p, s);
#endif
#ifndef PF_ONLY_N
    case 2048: return launch_col_mode<T, 2048, 8, PF_TP_2048>(mode, nslots, nbatch, p, s);
#endif
    }
    return cudaErrorInvalidValue;
}

template cudaError_t launch_col<double>(int, int, int, int, const ColParams<double> &, cudaStream_t);
template cudaError_t launch_col<float>(int, int, int, int, const ColParams<float> &, cudaStream_t);

}  // namespace pf
