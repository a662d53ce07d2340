// fft_core.cuh -- register/shared-memory Stockham FFT building blocks of libpf (product code; shares
// nothing with oracle/).
//
// One length-N complex transform is carried by TT = N/E cooperating threads; thread j holds the E
// elements  j + q*TT  (q = 0..E-1) in registers, BOTH before and after the transform (natural order
// on both sides), so pointwise work between transforms (the spectral update of Eqs. 14-15,
// PAPER.md:112-116, the Hermitian pack/unpack) needs no data movement.  A transform is a sequence of
// radix-R stages (R <= E, R a power of two): stage s with NS = product of the earlier radices computes,
// for every butterfly index jv in [0, N/R),
//     a[r] = in[jv + r*N/R] * W_{NS*R}^{r*(jv mod NS)},   a <- DFT_R(a),   out[(jv - jv mod NS)*R + jv mod NS + r*NS] = a[r]
// (Stockham autosort, decimation in time).  Between stages the data crosses shared memory once; the
// first stage reads and the last stage writes the register layout above, so a transform touches
// shared memory (stages-1) times.  Twiddles W_N^i come from a table (never sincos); powers within a
// butterfly are formed by a balanced product tree from one table load.
//
// Everything here is __host__ __device__ so that tests/test_fft_core_host.py can run the index logic
// on the CPU (thread loops emulated phase by phase).
#pragma once
#include <cuda_runtime.h>

#define PF_HD __host__ __device__ __forceinline__

namespace pf {

template <typename T> struct V2;
template <> struct V2<double> { typedef double2 type; };
template <> struct V2<float>  { typedef float2  type; };

template <typename T> PF_HD typename V2<T>::type mk(T x, T y) { typename V2<T>::type r; r.x = x; r.y = y; return r; }

template <typename C> PF_HD C cadd(C a, C b) { C r; r.x = a.x + b.x; r.y = a.y + b.y; return r; }
template <typename C> PF_HD C csub(C a, C b) { C r; r.x = a.x - b.x; r.y = a.y - b.y; return r; }
template <typename C> PF_HD C cmul(C a, C b) { C r; r.x = a.x * b.x - a.y * b.y; r.y = a.x * b.y + a.y * b.x; return r; }
template <typename C> PF_HD C csqr(C a)      { C r; r.x = (a.x - a.y) * (a.x + a.y); r.y = (a.x + a.x) * a.y; return r; }
template <typename C> PF_HD C cconj(C a)     { C r; r.x = a.x; r.y = -a.y; return r; }
template <typename C> PF_HD C cmul_mi(C a)   { C r; r.x = a.y; r.y = -a.x; return r; }   // a * (-i)
template <typename C> PF_HD C cmul_pi(C a)   { C r; r.x = -a.y; r.y = a.x; return r; }   // a * (+i)
template <typename C> PF_HD C cswap(C a)     { C r; r.x = a.y; r.y = a.x; return r; }
template <typename C, typename T> PF_HD C cscale(C a, T s) { C r; r.x = a.x * s; r.y = a.y * s; return r; }

// cos(m*pi/16) for any integer m, from the nine first-quadrant values (m = 0..8).
__host__ __device__ constexpr double cos_pi16_q(int m)
{
    return m == 0 ? 1.0
         : m == 1 ? 0.98078528040323044912618223613423903697393373089333609500291
         : m == 2 ? 0.92387953251128675612818318939678828682241662586364248611509
         : m == 3 ? 0.83146961230254523707878837761790575673856081198724243845118
         : m == 4 ? 0.70710678118654752440084436210484903928483593768847403658834
         : m == 5 ? 0.55557023301960222474283081394853287437493719075480404592415
         : m == 6 ? 0.38268343236508977172845998403039886676134456248562704143380
         : m == 7 ? 0.19509032201612826784828486847702224092769161775195480775450
         : 0.0;
}
__host__ __device__ constexpr double cos_pi16(int m)
{
    m = ((m % 32) + 32) % 32;                       // period 2*pi
    if (m > 16) m = 32 - m;                          // cos(2pi - x) = cos x
    return (m <= 8) ? cos_pi16_q(m) : -cos_pi16_q(16 - m);
}
__host__ __device__ constexpr double sin_pi16(int m) { return cos_pi16(m - 8); }

// a * W_R^k, W_R = exp(-2 pi i / R), R <= 32, as compile-time constants
template <int R, int K, typename C> PF_HD C cmul_wconst(C a)
{
    constexpr int m = (32 / R) * K;                  // angle = m*pi/16
    if (m % 32 == 0) return a;
    if (m % 32 == 8) return cmul_mi(a);
    if (m % 32 == 16) { C r; r.x = -a.x; r.y = -a.y; return r; }
    if (m % 32 == 24) return cmul_pi(a);
    typedef decltype(a.x) T;
    constexpr T c = (T)cos_pi16(m), s = (T)sin_pi16(m);   // W = c - i s
    C r; r.x = a.x * c + a.y * s; r.y = a.y * c - a.x * s; return r;
}

// DFT_R in place, natural order in and out, forward sign.
template <int R> struct Dft;
template <> struct Dft<1> { template <typename C> static PF_HD void run(C *) {} };
template <> struct Dft<2> {
    template <typename C> static PF_HD void run(C *a) { C t = a[0]; a[0] = cadd(t, a[1]); a[1] = csub(t, a[1]); }
};
template <> struct Dft<4> {
    template <typename C> static PF_HD void run(C *a)
    {
        C t0 = cadd(a[0], a[2]), t1 = csub(a[0], a[2]), t2 = cadd(a[1], a[3]), t3 = cmul_mi(csub(a[1], a[3]));
        a[0] = cadd(t0, t2); a[1] = cadd(t1, t3); a[2] = csub(t0, t2); a[3] = csub(t1, t3);
    }
};
template <int R, int K> struct DftCombine {
    template <typename C> static PF_HD void run(C *a, const C *e, const C *o)
    {
        C t = cmul_wconst<R, K>(o[K]);
        a[K] = cadd(e[K], t); a[K + R / 2] = csub(e[K], t);
        DftCombine<R, K + 1>::run(a, e, o);
    }
};
template <int R> struct DftCombine<R, R / 2> { template <typename C> static PF_HD void run(C *, const C *, const C *) {} };
template <int R> struct Dft {
    template <typename C> static PF_HD void run(C *a)
    {
        C e[R / 2], o[R / 2];
#pragma unroll
        for (int k = 0; k < R / 2; ++k) { e[k] = a[2 * k]; o[k] = a[2 * k + 1]; }
        Dft<R / 2>::run(e); Dft<R / 2>::run(o);
        DftCombine<R, 0>::run(a, e, o);
    }
};

// radix of the stage that starts with NS = product of the earlier radices
__host__ __device__ constexpr int stage_radix(int N, int E, int NS) { return (N / NS < E) ? N / NS : E; }
__host__ __device__ constexpr int num_stages(int N, int E) { int s = 0; for (int ns = 1; ns < N; ns *= stage_radix(N, E, ns)) ++s; return s; }

// First twiddle W_{NS*R}^{k} of each of the S = E/R butterflies thread j owns in the stage that starts at NS
// (k = butterfly index mod NS). Separated from the arithmetic so that a kernel can issue these table loads
// ahead of the barrier that precedes the stage. tw[i] = exp(-2 pi i * i / N), i in [0, N).
template <int N, int E, int NS> struct StageShape {
    static constexpr int R = stage_radix(N, E, NS);
    static constexpr int S = E / R;                   // butterflies per thread
    static constexpr int TT = N / E;
};
// TWS: tw points to shared memory (plain loads) instead of global memory (read-only path)
template <int N, int E, int NS, typename C, bool TWS = false>
PF_HD void stage_twiddles(C (&w1)[StageShape<N, E, NS>::S], int j, const C *__restrict__ tw)
{
    typedef StageShape<N, E, NS> Sh;
    if (NS > 1) {
#pragma unroll
        for (int m = 0; m < Sh::S; ++m) {
            const int k = (j + m * Sh::TT) & (NS - 1);
#if defined(__CUDA_ARCH__)
            if (TWS) w1[m] = tw[k * (N / (NS * Sh::R))];
            else w1[m] = __ldg(tw + k * (N / (NS * Sh::R)));
#else
            w1[m] = tw[k * (N / (NS * Sh::R))];
#endif
        }
    }
}

// twiddle + butterflies of one stage on the E registers of a thread (see the header comment); w1 from stage_twiddles.
// Powers within a butterfly are formed by a balanced product tree.
template <int N, int E, int NS, typename C>
PF_HD void stage_compute_w(C (&v)[E], const C (&w1)[StageShape<N, E, NS>::S])
{
#ifdef PF_DBG_SKIP_COMPUTE
    return;
#endif
    constexpr int R = StageShape<N, E, NS>::R;
    constexpr int S = StageShape<N, E, NS>::S;
#pragma unroll
    for (int m = 0; m < S; ++m) {
        C a[R];
#pragma unroll
        for (int r = 0; r < R; ++r) a[r] = v[m + r * S];
        if (NS > 1) {
            C w[R];
            w[1] = w1[m];
#pragma unroll
            for (int r = 2; r < R; ++r) w[r] = (r & 1) ? cmul(w[r / 2], w[r - r / 2]) : csqr(w[r / 2]);
#pragma unroll
            for (int r = 1; r < R; ++r) a[r] = cmul(a[r], w[r]);
        }
        Dft<R>::run(a);
#pragma unroll
        for (int r = 0; r < R; ++r) v[m + r * S] = a[r];
    }
}

// twiddle + butterflies of one stage on the E registers of thread j (table load at the point of use)
template <int N, int E, int NS, typename C>
PF_HD void stage_compute(C (&v)[E], int j, const C *__restrict__ tw)
{
    C w1[StageShape<N, E, NS>::S];
    stage_twiddles<N, E, NS>(w1, j, tw);
    stage_compute_w<N, E, NS>(v, w1);
}

// scatter the outputs of a non-final stage into the exchange buffer; buf(i) -> reference to element i
template <int N, int E, int NS, typename C, typename Buf>
PF_HD void exchange_store(const C (&v)[E], int j, Buf &buf)
{
#ifdef PF_DBG_SKIP_EXCHANGE
    return;
#endif
    constexpr int R = stage_radix(N, E, NS);
    constexpr int S = E / R;
    constexpr int TT = N / E;
#pragma unroll
    for (int m = 0; m < S; ++m) {
        const int jv = j + m * TT;
        const int k = jv & (NS - 1);
        const int j0 = (jv - k) * R + k;
#pragma unroll
        for (int r = 0; r < R; ++r) buf.st(j0 + r * NS, v[m + r * S]);
    }
}
template <int N, int E, typename C, typename Buf>
PF_HD void exchange_load(C (&v)[E], int j, const Buf &buf)
{
#ifdef PF_DBG_SKIP_EXCHANGE
    return;
#endif
    constexpr int TT = N / E;
#pragma unroll
    for (int q = 0; q < E; ++q) v[q] = buf.ld(j + q * TT);
}

#if defined(__CUDACC__)
// Full forward transform of one column held by the TT threads that share `buf`; sync() must be a barrier over (at
// least) those threads. Inverse = swap re/im, forward, swap re/im (unnormalised). Buf provides
// store<N, E, NS>(v, j) (Stockham scatter of a non-final stage) and load<N, E>(v, j) (elements j + q*TT).
// w1 = twiddles of the stage that starts at NS; those of the next stage are requested between the two barriers
// of the exchange, when the data registers are dead and the table latency hides behind the barrier.
//
// Pol is the execution policy of the group of threads that carries the transform:
//   barrier()        barrier over (at least) the TT threads that share `buf`;
//   begin_compute()  called before the butterflies of every stage, end_compute() after the barrier that follows the
//                    butterflies of every stage but the last (the caller keeps computing after the last stage and ends
//                    the phase itself). No-ops except where thread groups of an SM take turns on the fp64 pipe
//                    (col2d_kernels.cu).
template <typename Sync> struct SyncOnly {
    const Sync &sync;
    __device__ __forceinline__ void barrier() const { sync(); }
    __device__ __forceinline__ void begin_compute() const {}
    __device__ __forceinline__ void end_compute() const {}
};
template <int N, int E, int NS, bool TWS, typename C, typename Buf, typename Pol>
__device__ __forceinline__ void fft_stages_p(C (&v)[E], int j, const C *__restrict__ tw, Buf &buf, Pol &pol,
                                             const C (&w1)[StageShape<N, E, NS>::S])
{
    pol.begin_compute();
    stage_compute_w<N, E, NS>(v, w1);
    constexpr int R = stage_radix(N, E, NS);
    if constexpr (NS * R < N) {
        C w2[StageShape<N, E, NS * R>::S];
        pol.barrier();                            // every thread has taken its elements of the previous exchange
        pol.end_compute();
#ifndef PF_DBG_SKIP_EXCHANGE
        buf.template store<N, E, NS>(v, j);
#endif
#ifndef PF_NO_TW_HOIST
        stage_twiddles<N, E, NS * R, C, TWS>(w2, j, tw);
#endif
        pol.barrier();
#ifdef PF_NO_TW_HOIST
        stage_twiddles<N, E, NS * R, C, TWS>(w2, j, tw);
#endif
#ifndef PF_DBG_SKIP_EXCHANGE
        buf.template load<N, E>(v, j);
#endif
        fft_stages_p<N, E, NS * R, TWS>(v, j, tw, buf, pol, w2);
    }
}
template <int N, int E, bool TWS = false, typename C, typename Buf, typename Pol>
__device__ __forceinline__ void fft_forward_p(C (&v)[E], int j, const C *__restrict__ tw, Buf &buf, Pol &pol)
{
    C w0[StageShape<N, E, 1>::S];                 // the first stage has no twiddles; never read
    fft_stages_p<N, E, 1, TWS>(v, j, tw, buf, pol, w0);
}
template <int N, int E, bool TWS = false, typename C, typename Buf, typename Sync>
__device__ __forceinline__ void fft_forward(C (&v)[E], int j, const C *__restrict__ tw, Buf &buf, const Sync &sync)
{
    SyncOnly<Sync> pol{sync};
    fft_forward_p<N, E, TWS>(v, j, tw, buf, pol);
}
template <int E, typename C> __device__ __forceinline__ void swap_all(C (&v)[E])
{
#pragma unroll
    for (int q = 0; q < E; ++q) v[q] = cswap(v[q]);
}
#endif

}  // namespace pf
