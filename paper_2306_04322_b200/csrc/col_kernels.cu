// col_kernels.cu -- strided-direction kernels of the Fourier-spectral step.
//
// A CTA owns TP "units" of two columns each and all N elements of them along the FFT axis; thread
// (t, j) holds elements j + q*TT of both columns of unit t in registers (fft_core.cuh) and the two
// transforms run interleaved. Consecutive lanes map to consecutive columns, so every global access of
// a warp is made of contiguous 16*TP-byte (fp64) pieces, and the strided "transpose" happens in
// registers + one shared-memory exchange per FFT stage boundary.
//
// Units in the pair modes are the mirror pairs (k, M-k) of the z-form (row_kernels.cu): with
//   E = (Z_k + conj Z_{M-k})/2,  O = -(i/2)(Z_k - conj Z_{M-k}),  W = exp(-2 pi i k / nx)
// the true half-spectrum columns are  U_k = E + W O  and  U_{M-k} = conj(E - W O), pointwise along the
// column; k = 0 yields the DC and Nyquist columns from Z_0 alone and k = M/2 is its own mirror. The
// inverse relations repack two updated columns into z-form. The spectral update itself is
//   c^   <- ( c^ - dt M |xi|^2 g^ ) / ( 1 + dt M kappa_c |xi|^4 )        Eqs. 12, 14
//   eta^ <- w^ / ( 1 + dt L kappa_eta |xi|^2 ),  w = eta - dt L h        Eqs. 13, 15
// with |xi|^2 = kx2 + ky2 (+ kz2) from 1-D tables (Eq. 16/19 or the FS-FD variants).
#include "pf_kernels.cuh"

namespace pf {

template <typename C, int STRIDE> struct ColBuf {
    C *base;
    __device__ __forceinline__ void st(int i, C v) { base[i * STRIDE] = v; }
    __device__ __forceinline__ C ld(int i) const { return base[i * STRIDE]; }
};
struct CtaSync2 { __device__ __forceinline__ void operator()() const { __syncthreads(); } };

template <typename T, int N, int E, int TP, int MODE, bool IS_C>
__global__ void __launch_bounds__(TP *(N / E)) col_kernel(const ColParams<T> p)
{
    typedef typename V2<T>::type C;
    constexpr int TT = N / E;
    constexpr bool PAIR_IN = (MODE == COL_2D_LAST || MODE == COL_3D_MIDFWD || MODE == COL_2D_ENERGY);
    constexpr bool PAIR_OUT = (MODE == COL_2D_LAST || MODE == COL_3D_MIDINV);
    constexpr bool ENERGY = (MODE == COL_2D_ENERGY || MODE == COL_3D_ENERGY);
    constexpr bool DO_FWD = (MODE != COL_3D_MIDINV);
    constexpr bool DO_UPD = (MODE == COL_2D_LAST || MODE == COL_3D_LAST);
    constexpr bool DO_INV = (MODE == COL_2D_LAST || MODE == COL_3D_LAST || MODE == COL_3D_MIDINV);
    constexpr bool LAST3D = (MODE == COL_3D_LAST || MODE == COL_3D_ENERGY);
    constexpr int SLOTS = 2 * TP;

    extern __shared__ __align__(16) unsigned char smem_raw[];
    C *xbuf = reinterpret_cast<C *>(smem_raw);
    C *stash = xbuf + N * SLOTS;                       // IS_C only

    const int t = threadIdx.x % TP;
    const int j = threadIdx.x / TP;
    const int M = p.M;
    const long fz = blockIdx.z, bz = blockIdx.y;

    // ---- which two columns ----
    bool valid, storeB;
    int zcolA = 0, zcolB = 0;            // column indices in z-form arrays (pitch M)
    int pcolA, pcolB;                     // column indices in plain arrays
    int kxA, kxB;                         // kx of the two columns
    T base2A, base2B;                     // |xi|^2 contributions that are constant along the column
    C wx = mk<T>(1, 0);                   // exp(-2 pi i u / nx)
    if (PAIR_IN || PAIR_OUT) {
        int u = blockIdx.x * TP + t;
        valid = (u <= M / 2);
        if (!valid) u = 0;
        zcolA = u; zcolB = (M - u) & (M - 1);
        kxA = u; kxB = M - u;
        pcolA = kxA; pcolB = kxB;
        storeB = valid && (kxB != kxA) ;
        wx = p.twx[u];
        base2A = p.kx2[kxA]; base2B = p.kx2[kxB];
    } else {
        pcolA = blockIdx.x * SLOTS + t; pcolB = pcolA + TP;
        valid = pcolB < p.ncols;                       // ncols is a multiple of SLOTS
        if (!valid) { pcolA = t; pcolB = TP + t; }
        storeB = valid;
        kxA = pcolA % p.P2; kxB = pcolB % p.P2;
        base2A = p.kx2[kxA] + p.ky2[pcolA / p.P2];
        base2B = p.kx2[kxB] + p.ky2[pcolB / p.P2];
    }
    const T *klast = LAST3D ? p.kz2 : p.ky2;

    ColBuf<C, SLOTS> bufA{xbuf + t}, bufB{xbuf + TP + t};
    CtaSync2 sync;

    auto load_pair = [&](const C *src, C(&va)[E], C(&vb)[E]) {
        if (PAIR_IN) {
#pragma unroll
            for (int q = 0; q < E; ++q) {
                const long i = j + q * TT;
                const C za = src[i * p.in_rs + zcolA], zb = src[i * p.in_rs + zcolB];
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
                va[q] = src[i * p.in_rs + pcolA];
                vb[q] = src[i * p.in_rs + pcolB];
            }
        }
    };

    C va[E], vb[E];
    const C *in0 = p.in0 + fz * p.in_fs + bz * p.in_bs;

    if (IS_C && DO_UPD) {
        // g first: transform and park it in thread-private shared-memory slots
        const C *in1 = p.in1 + fz * p.in1_fs + bz * p.in_bs;
        load_pair(in1, va, vb);
        fft2_stages<N, E, 1>(va, vb, j, p.tw, bufA, bufB, sync);
#pragma unroll
        for (int q = 0; q < E; ++q) {
            stash[(q * 2 + 0) * (TP * TT) + threadIdx.x] = va[q];
            stash[(q * 2 + 1) * (TP * TT) + threadIdx.x] = vb[q];
        }
    }

    load_pair(in0, va, vb);
    if (DO_FWD) fft2_stages<N, E, 1>(va, vb, j, p.tw, bufA, bufB, sync);

    if (DO_UPD) {
        const T s = T(1) / T(N);
#pragma unroll
        for (int q = 0; q < E; ++q) {
            const T kl = klast[j + q * TT];
            const T k2a = base2A + kl, k2b = base2B + kl;
            if (IS_C) {
                const C ga = stash[(q * 2 + 0) * (TP * TT) + threadIdx.x];
                const C gb = stash[(q * 2 + 1) * (TP * TT) + threadIdx.x];
                const T da = s / (T(1) + p.m.dtMkc * k2a * k2a), db = s / (T(1) + p.m.dtMkc * k2b * k2b);
                const T ma = p.m.dtM * k2a, mb = p.m.dtM * k2b;
                va[q] = mk<T>((va[q].x - ma * ga.x) * da, (va[q].y - ma * ga.y) * da);
                vb[q] = mk<T>((vb[q].x - mb * gb.x) * db, (vb[q].y - mb * gb.y) * db);
            } else {
                const T da = s / (T(1) + p.m.dtLke * k2a), db = s / (T(1) + p.m.dtLke * k2b);
                va[q] = cscale(va[q], da);
                vb[q] = cscale(vb[q], db);
            }
        }
    }

    if (ENERGY) {
        // sum over the full spectrum of |xi|^2 |u^|^2: columns with 0 < kx < M stand for their mirror too
        double acc = 0.0;
        const double wa = (kxA == 0 || kxA == M) ? 1.0 : 2.0, wb = (kxB == 0 || kxB == M) ? 1.0 : 2.0;
        const bool useA = valid && kxA <= M, useB = storeB && kxB <= M;
#pragma unroll
        for (int q = 0; q < E; ++q) {
            const T kl = klast[j + q * TT];
            if (useA) acc += wa * (double)(base2A + kl) * ((double)va[q].x * va[q].x + (double)va[q].y * va[q].y);
            if (useB) acc += wb * (double)(base2B + kl) * ((double)vb[q].x * vb[q].x + (double)vb[q].y * vb[q].y);
        }
        double *red = reinterpret_cast<double *>(smem_raw);      // off the hot path: plain serial reduction
        sync();
        red[threadIdx.x] = acc;
        sync();
        if (threadIdx.x == 0) {
            double tot = 0.0;
            for (int w = 0; w < TP * TT; ++w) tot += red[w];
            atomicAdd(p.acc + fz, tot);
        }
        return;
    }

    if (DO_INV) {
        swap_all(va); swap_all(vb);
        fft2_stages<N, E, 1>(va, vb, j, p.tw, bufA, bufB, sync);
        swap_all(va); swap_all(vb);
        if (!DO_UPD) {                                   // mid inverse: normalise here (update folds 1/N in)
            const T s = T(1) / T(N);
#pragma unroll
            for (int q = 0; q < E; ++q) { va[q] = cscale(va[q], s); vb[q] = cscale(vb[q], s); }
        }
    }

    C *out = p.out + fz * p.out_fs + bz * p.out_bs;
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

template <typename T, int N, int E, int TP, int MODE, bool IS_C>
static cudaError_t launch_col_inst(int nfields, int nbatch, const ColParams<T> &p, cudaStream_t s)
{
    typedef typename V2<T>::type C;
    constexpr int TT = N / E;
    constexpr bool PAIRS = (MODE == COL_2D_LAST || MODE == COL_3D_MIDFWD || MODE == COL_3D_MIDINV || MODE == COL_2D_ENERGY);
    const int ntiles = PAIRS ? (p.M / 2 + 1 + TP - 1) / TP : (p.ncols + 2 * TP - 1) / (2 * TP);
    size_t smem = (size_t)N * 2 * TP * sizeof(C) * ((IS_C && (MODE == COL_2D_LAST || MODE == COL_3D_LAST)) ? 2 : 1);
    auto kern = col_kernel<T, N, E, TP, MODE, IS_C>;
    if (smem > 48 * 1024) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
    }
    dim3 grid((unsigned)ntiles, (unsigned)nbatch, (unsigned)nfields);
    kern<<<grid, TP * TT, smem, s>>>(p);
    return cudaGetLastError();
}

template <typename T, int N, int E, int TP>
static cudaError_t launch_col_mode(int mode, bool is_c, int nfields, int nbatch, const ColParams<T> &p, cudaStream_t s)
{
    switch (mode) {
    case COL_2D_LAST:
        return is_c ? launch_col_inst<T, N, E, TP, COL_2D_LAST, true>(nfields, nbatch, p, s)
                    : launch_col_inst<T, N, E, TP, COL_2D_LAST, false>(nfields, nbatch, p, s);
    case COL_3D_MIDFWD: return launch_col_inst<T, N, E, TP, COL_3D_MIDFWD, false>(nfields, nbatch, p, s);
    case COL_3D_MIDINV: return launch_col_inst<T, N, E, TP, COL_3D_MIDINV, false>(nfields, nbatch, p, s);
    case COL_3D_LAST:
        return is_c ? launch_col_inst<T, N, E, TP, COL_3D_LAST, true>(nfields, nbatch, p, s)
                    : launch_col_inst<T, N, E, TP, COL_3D_LAST, false>(nfields, nbatch, p, s);
    case COL_2D_ENERGY: return launch_col_inst<T, N, E, TP, COL_2D_ENERGY, false>(nfields, nbatch, p, s);
    case COL_3D_ENERGY: return launch_col_inst<T, N, E, TP, COL_3D_ENERGY, false>(nfields, nbatch, p, s);
    }
    return cudaErrorInvalidValue;
}

// nfft = length of the FFT axis. Column-pair units per CTA: enough threads per CTA for small N,
// shared memory <= ~64 KB per CTA for large N.
template <typename T> cudaError_t launch_col(int mode, bool is_c, int nfft, int nfields, int nbatch,
                                             const ColParams<T> &p, cudaStream_t s)
{
    switch (nfft) {
    case 16:   return launch_col_mode<T, 16, 8, 8>(mode, is_c, nfields, nbatch, p, s);
    case 32:   return launch_col_mode<T, 32, 8, 8>(mode, is_c, nfields, nbatch, p, s);
    case 64:   return launch_col_mode<T, 64, 8, 8>(mode, is_c, nfields, nbatch, p, s);
    case 128:  return launch_col_mode<T, 128, 8, 8>(mode, is_c, nfields, nbatch, p, s);
    case 256:  return launch_col_mode<T, 256, 8, 4>(mode, is_c, nfields, nbatch, p, s);
    case 512:  return launch_col_mode<T, 512, 8, 4>(mode, is_c, nfields, nbatch, p, s);
    case 1024: return launch_col_mode<T, 1024, 8, 2>(mode, is_c, nfields, nbatch, p, s);
    case 2048:
        // the c-field variant parks g^ in a second buffer: one unit per CTA keeps it within 227 KB
        return is_c ? launch_col_mode<T, 2048, 16, 1>(mode, is_c, nfields, nbatch, p, s)
                    : launch_col_mode<T, 2048, 16, 2>(mode, is_c, nfields, nbatch, p, s);
    }
    return cudaErrorInvalidValue;
}

template cudaError_t launch_col<double>(int, bool, int, int, int, const ColParams<double> &, cudaStream_t);
template cudaError_t launch_col<float>(int, bool, int, int, int, const ColParams<float> &, cudaStream_t);

}  // namespace pf
