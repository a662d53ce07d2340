// col_kernels.cu -- strided-direction kernels of the Fourier-spectral step.
//
// A CTA is two independent thread GROUPS; a group owns TP "units" of two columns each and all N elements of
// them along the FFT axis; thread (t, j) of a group holds elements j + q*TT of both columns of unit t in
// registers (fft_core.cuh) and the two transforms run half a stage out of phase (fft2_pipelined).
// Consecutive lanes map to consecutive columns, so every global access of a warp is made of contiguous
// 16*TP-byte (fp64) pieces, and the strided "transpose" happens in registers + one shared-memory exchange
// per FFT stage boundary. Groups synchronise only through their own mbarriers, so the two groups of a CTA
// (and the CTAs of an SM) drift apart and overlap each other's memory, shared-memory and fp64 phases.
//
// Units in the pair modes are the mirror pairs (k, M-k) of the z-form (row_kernels.cu): with
//   E = (Z_k + conj Z_{M-k})/2,  O = -(i/2)(Z_k - conj Z_{M-k}),  W = exp(-2 pi i k / nx)
// the true half-spectrum columns are  U_k = E + W O  and  U_{M-k} = conj(E - W O), pointwise along the
// column; k = 0 yields the DC and Nyquist columns from Z_0 alone and k = M/2 is its own mirror. The
// inverse relations repack two updated columns into z-form. The spectral update itself is
//   c^   <- ( c^ - dt M |xi|^2 g^ ) / ( 1 + dt M kappa_c |xi|^4 )        Eqs. 12, 14
//   eta^ <- w^ / ( 1 + dt L kappa_eta |xi|^2 ),  w = eta - dt L h        Eqs. 13, 15
// with |xi|^2 = kx2 + ky2 (+ kz2) from 1-D tables (Eq. 16/19 or the FS-FD variants).
//
// Field slots (blockIdx.z): in the update modes slot 0 is c, whose CTA uses its two groups for the two arrays
// the update needs on the SAME units: group 0 transforms g = df/dc, scales it by dt M |xi|^2 and hands it over
// through shared memory; group 1 transforms c^, combines, inverts and stores. Every other CTA uses its two
// groups for two consecutive blocks of units of one array.
#include "pf_kernels.cuh"

namespace pf {

// Exchange buffer of a group: N rows (index along the FFT axis) x 2*TP column slots (slot = side*TP + t) of one
// complex each. A quarter warp (8 lanes x 16 B, one shared-memory wavefront when conflict free) covers 8/TP
// different rows; which rows depends on the access: consecutive rows for the loads (j + q*TT) and for the stores
// of later stages, rows R apart for the stores of the first stage. The placement below XORs the position of a
// row's slots inside its 128-byte line with parities of the row index taken over the bit sets
// {b, b+LR, b+2LR, ..} (LR = log2 of the first-stage radix), which flip under either pattern.
template <typename C, int TP, int LR> struct ColBuf {
    C *base;          // buffer start
    int side, t;      // this thread's column slot
    __device__ __forceinline__ static int par(int row, int b)
    {
        unsigned m = 0;
#pragma unroll
        for (int k = b; k < 12; k += LR) m |= 1u << k;
        return __popc((unsigned)row & m) & 1;
    }
    __device__ __forceinline__ int idx(int row) const
    {
        if (TP == 4) return row * 8 + ((side ^ par(row, 0)) * 4 + t);                            // line = 1 row
        if (TP == 2) return (row >> 1) * 8 + (2 * par(row, 0) + (side ^ par(row, 1))) * 2 + t;   // line = 2 rows
        return row * (2 * TP) + side * TP + t;
    }
    __device__ __forceinline__ void st(int i, C v) { base[idx(i)] = v; }
    __device__ __forceinline__ C ld(int i) const { return base[idx(i)]; }
};

__device__ __forceinline__ double rcp(double x) { return __drcp_rn(x); }
__device__ __forceinline__ float rcp(float x) { return __frcp_rn(x); }

template <typename T, int N, int E, int TP, int MODE>
__global__ void __launch_bounds__(2 * TP *(N / E), (2 * TP * (N / E) >= 512) ? 1 : 512 / (2 * TP * (N / E)))
col_kernel(const ColParams<T> p)
{
#ifdef PF_DBG_EMPTY
    return;
#endif
    typedef typename V2<T>::type C;
    constexpr int TT = N / E;
    constexpr int GT = TP * TT;                        // threads per group (a multiple of 32)
    constexpr bool PAIRS = (MODE == COL_2D_LAST || MODE == COL_3D_MIDFWD || MODE == COL_3D_MIDINV || MODE == COL_2D_ENERGY);
    constexpr bool PAIR_IN = (MODE == COL_2D_LAST || MODE == COL_3D_MIDFWD || MODE == COL_2D_ENERGY);
    constexpr bool PAIR_OUT = (MODE == COL_2D_LAST || MODE == COL_3D_MIDINV);
    constexpr bool ENERGY = (MODE == COL_2D_ENERGY || MODE == COL_3D_ENERGY);
    constexpr bool DO_FWD = (MODE != COL_3D_MIDINV);
    constexpr bool DO_UPD = (MODE == COL_2D_LAST || MODE == COL_3D_LAST);
    constexpr bool DO_INV = (MODE == COL_2D_LAST || MODE == COL_3D_LAST || MODE == COL_3D_MIDINV);
    constexpr bool LAST3D = (MODE == COL_3D_LAST || MODE == COL_3D_ENERGY);
    constexpr int SLOTS = 2 * TP;
    constexpr int LR = (E >= 16) ? 4 : 3;
    static_assert(GT % 32 == 0, "a group must be whole warps");

    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int g = threadIdx.x / GT;                    // group
    const int tg = threadIdx.x - g * GT;
    const int t = tg % TP;
    const int j = tg / TP;
    const int M = p.M;
    const int slot = blockIdx.z;
    const long bz = blockIdx.y;
    const bool c_cta = DO_UPD && p.has_c && slot == 0;

    C *xbuf = reinterpret_cast<C *>(smem_raw) + (long)g * N * SLOTS;
    PipeBars bars;
    bars.init(smem_raw + p.bar_off + 32 * g, GT / 32, tg == 0);
    __syncthreads();

    // ---- which block of units, which two columns ----
    const int nblk = PAIRS ? (M / 2 + TP) / TP : p.ncols / SLOTS;
    const int ub = c_cta ? (int)blockIdx.x : 2 * (int)blockIdx.x + g;
    bool valid = ub < nblk;
    bool storeB;
    int zcolA = 0, zcolB = 0;             // column indices in z-form arrays (pitch M)
    int pcolA, pcolB;                     // column indices in plain arrays
    int kxA, kxB;                         // kx of the two columns
    T base2A, base2B;                     // |xi|^2 contributions that are constant along the column
    C wx = mk<T>(1, 0);                   // exp(-2 pi i u / nx)
    if (PAIRS) {
        int u = ub * TP + t;
        valid = valid && (u <= M / 2);
        if (!valid) u = 0;
        zcolA = u; zcolB = (M - u) & (M - 1);
        kxA = u; kxB = M - u;
        pcolA = kxA; pcolB = kxB;
        storeB = valid && (kxB != kxA);
        wx = p.twx[u];
        base2A = p.kx2[kxA]; base2B = p.kx2[kxB];
    } else {
        pcolA = (valid ? ub : 0) * SLOTS + t; pcolB = pcolA + TP;
        storeB = valid;
        kxA = pcolA % p.P2; kxB = pcolB % p.P2;
        base2A = p.kx2[kxA] + p.ky2[pcolA / p.P2];
        base2B = p.kx2[kxB] + p.ky2[pcolB / p.P2];
    }
    // a CTA whose two groups both have no units leaves (eta slots are launched with the c slot's grid)
    if (!ENERGY && __syncthreads_or(valid) == 0) return;
    const T *klast = LAST3D ? p.kz2 : p.ky2;
    T kl[E];
    if (DO_UPD || ENERGY) {
#pragma unroll
        for (int q = 0; q < E; ++q) kl[q] = klast[j + q * TT];       // constant tables: issued early
    }

    // ---- arrays of this CTA / group ----
    const C *in;
    C *out;
    if (c_cta) {
        in = (g == 0) ? p.in1 : p.in0;
        out = p.out;
    } else if (slot == 0 && p.alt_in) {
        in = p.alt_in; out = p.alt_out;
    } else {
        in = p.in0 + slot * p.in_fs;
        out = p.out + slot * p.out_fs;
    }
    in += bz * p.in_bs;
    out += bz * p.out_bs;

    ColBuf<C, TP, LR> bufA{xbuf, 0, t}, bufB{xbuf, 1, t};
    C va[E], vb[E];

    grid_dependency_wait();                // everything above touches constant tables only
    grid_dependents_launch();

    if (PAIR_IN) {
#pragma unroll
        for (int q = 0; q < E; ++q) {
            const long i = j + q * TT;
            const C za = in[i * p.in_rs + zcolA], zb = in[i * p.in_rs + zcolB];
            // E = (za + conj zb)/2, O = -(i/2)(za - conj zb)
            const C e = mk<T>(T(0.5) * (za.x + zb.x), T(0.5) * (za.y - zb.y));
            const C o = mk<T>(T(0.5) * (za.y + zb.y), T(-0.5) * (za.x - zb.x));
            const C wo = cmul(wx, o);
            va[q] = cadd(e, wo);
            vb[q] = cconj(csub(e, wo));
        }
    } else {
#pragma unroll
        for (int q = 0; q < E; ++q) {
            const long i = j + q * TT;
            va[q] = in[i * p.in_rs + pcolA];
            vb[q] = in[i * p.in_rs + pcolB];
        }
    }

    if (DO_FWD) fft2_pipelined<N, E, 1, true>(va, vb, j, p.tw, bufA, bufB, bars);

#ifndef PF_DBG_SKIP_UPDATE
    if (DO_UPD) {
        const T s = T(1) / T(N);
        if (c_cta) {
            // group 0: dt M |xi|^2 g^ -> shared memory (thread-linear in its own buffer) -> group 1
            C *hand = reinterpret_cast<C *>(smem_raw);
            if (g == 0) {
                asm volatile("bar.sync 1, %0;" ::"r"(GT) : "memory");       // group 0 has left its exchange buffer
#pragma unroll
                for (int q = 0; q < E; ++q) {
                    const T ma = p.m.dtM * (base2A + kl[q]), mb = p.m.dtM * (base2B + kl[q]);
                    hand[(q * 2 + 0) * GT + tg] = cscale(va[q], ma);
                    hand[(q * 2 + 1) * GT + tg] = cscale(vb[q], mb);
                }
            }
            __syncthreads();
            if (g == 0) return;
#pragma unroll
            for (int q = 0; q < E; ++q) {
                const T k2a = base2A + kl[q], k2b = base2B + kl[q];
                const T da = s * rcp(T(1) + p.m.dtMkc * k2a * k2a), db = s * rcp(T(1) + p.m.dtMkc * k2b * k2b);
                const C ga = hand[(q * 2 + 0) * GT + tg], gb = hand[(q * 2 + 1) * GT + tg];
                va[q] = mk<T>((va[q].x - ga.x) * da, (va[q].y - ga.y) * da);
                vb[q] = mk<T>((vb[q].x - gb.x) * db, (vb[q].y - gb.y) * db);
            }
        } else {
#pragma unroll
            for (int q = 0; q < E; ++q) {
                const T k2a = base2A + kl[q], k2b = base2B + kl[q];
                const T da = s * rcp(T(1) + p.m.dtLke * k2a), db = s * rcp(T(1) + p.m.dtLke * k2b);
                va[q] = cscale(va[q], da);
                vb[q] = cscale(vb[q], db);
            }
        }
    }
#endif

    if (ENERGY) {
        // sum over the full spectrum of |xi|^2 |u^|^2: columns with 0 < kx < M stand for their mirror too
        double acc = 0.0;
        const double wa = (kxA == 0 || kxA == M) ? 1.0 : 2.0, wb = (kxB == 0 || kxB == M) ? 1.0 : 2.0;
        const bool useA = valid && kxA <= M, useB = storeB && kxB <= M;
#pragma unroll
        for (int q = 0; q < E; ++q) {
            if (useA) acc += wa * (double)(base2A + kl[q]) * ((double)va[q].x * va[q].x + (double)va[q].y * va[q].y);
            if (useB) acc += wb * (double)(base2B + kl[q]) * ((double)vb[q].x * vb[q].x + (double)vb[q].y * vb[q].y);
        }
        double *red = reinterpret_cast<double *>(smem_raw);      // off the hot path: plain serial reduction
        __syncthreads();
        red[threadIdx.x] = acc;
        __syncthreads();
        if (threadIdx.x == 0) {
            double tot = 0.0;
            for (int w = 0; w < 2 * GT; ++w) tot += red[w];
            atomicAdd(p.acc + slot, tot);
        }
        return;
    }

    if (DO_INV) {
        swap_all(va); swap_all(vb);
        fft2_pipelined<N, E, 1, true>(va, vb, j, p.tw, bufA, bufB, bars);
        swap_all(va); swap_all(vb);
        if (!DO_UPD) {                                   // mid inverse: normalise here (the update folds 1/N in)
            const T s = T(1) / T(N);
#pragma unroll
            for (int q = 0; q < E; ++q) { va[q] = cscale(va[q], s); vb[q] = cscale(vb[q], s); }
        }
    }

    if (PAIR_OUT) {
        // E = (Ua + conj Ub)/2, W O = (Ua - conj Ub)/2, Z_a = E + i O, Z_b = conj(E - i O)
        const C wxc = cconj(wx);
#pragma unroll
        for (int q = 0; q < E; ++q) {
            const long i = j + q * TT;
            const C e = mk<T>(T(0.5) * (va[q].x + vb[q].x), T(0.5) * (va[q].y - vb[q].y));
            const C wo = mk<T>(T(0.5) * (va[q].x - vb[q].x), T(0.5) * (va[q].y + vb[q].y));
            const C o = cmul(wxc, wo);
            const C io = cmul_pi(o);
            if (valid) out[i * p.out_rs + zcolA] = cadd(e, io);
            if (storeB && zcolB != zcolA) out[i * p.out_rs + zcolB] = cconj(csub(e, io));
        }
    } else {
#pragma unroll
        for (int q = 0; q < E; ++q) {
            const long i = j + q * TT;
            if (valid) out[i * p.out_rs + pcolA] = va[q];
            if (storeB) out[i * p.out_rs + pcolB] = vb[q];
        }
    }
}

template <typename T, int N, int E, int TP, int MODE>
static cudaError_t launch_col_inst(int nslots, int nbatch, const ColParams<T> &p, cudaStream_t s)
{
    typedef typename V2<T>::type C;
    constexpr int TT = N / E;
    constexpr bool PAIRS = (MODE == COL_2D_LAST || MODE == COL_3D_MIDFWD || MODE == COL_3D_MIDINV || MODE == COL_2D_ENERGY);
    constexpr bool DO_UPD = (MODE == COL_2D_LAST || MODE == COL_3D_LAST);
    const int nblk = PAIRS ? (p.M / 2 + TP) / TP : p.ncols / (2 * TP);
    const int gx = (DO_UPD && p.has_c) ? nblk : (nblk + 1) / 2;       // a c CTA covers one block of units, the others two
    size_t smem = (size_t)2 * N * 2 * TP * sizeof(C);
    ColParams<T> q = p;
    q.bar_off = (int)smem;                   // 2 x 4 mbarriers behind the exchange buffers
    smem += 64;
    auto kern = col_kernel<T, N, E, TP, MODE>;
    if (smem > 48 * 1024) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
    }
    return launch_pdl(kern, dim3((unsigned)gx, (unsigned)nbatch, (unsigned)nslots), dim3(2 * TP * TT), smem, s, p.pdl != 0, q);
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

// nfft = length of the FFT axis. TP (units per group) keeps a group at whole warps for short axes and the two
// exchange buffers of a CTA within 128 KB for long ones.
template <typename T> cudaError_t launch_col(int mode, int nfft, int nslots, int nbatch, const ColParams<T> &p, cudaStream_t s)
{
    switch (nfft) {
#ifndef PF_ONLY_N
    case 16:   return launch_col_mode<T, 16, 8, 16>(mode, nslots, nbatch, p, s);
    case 32:   return launch_col_mode<T, 32, 8, 8>(mode, nslots, nbatch, p, s);
    case 64:   return launch_col_mode<T, 64, 8, 8>(mode, nslots, nbatch, p, s);
    case 128:  return launch_col_mode<T, 128, 8, 4>(mode, nslots, nbatch, p, s);
    case 256:  return launch_col_mode<T, 256, 8, 4>(mode, nslots, nbatch, p, s);
    case 512:  return launch_col_mode<T, 512, 8, 4>(mode, nslots, nbatch, p, s);
#endif
#if !defined(PF_ONLY_N) || PF_ONLY_N == 1024
    case 1024: return launch_col_mode<T, 1024, 8, 2>(mode, nslots, nbatch, p, s);
#endif
#ifndef PF_ONLY_N
    case 2048: return launch_col_mode<T, 2048, 16, 1>(mode, nslots, nbatch, p, s);
#endif
    }
    return cudaErrorInvalidValue;
}

template cudaError_t launch_col<double>(int, int, int, int, const ColParams<double> &, cudaStream_t);
template cudaError_t launch_col<float>(int, int, int, int, const ColParams<float> &, cudaStream_t);

}  // namespace pf
