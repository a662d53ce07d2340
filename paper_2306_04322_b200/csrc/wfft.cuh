// wfft.cuh -- "warp-tile" FFT of the strided kernels for the long axes (N = 256 .. 2048, 8 elements per thread): the
// product path's transform where one exchange per transform crosses shared memory and everything else stays inside a
// warp (shuffles). Product code; shares nothing with oracle/.
//
// A column of N = 64 * 2^HB points is carried by TT = N/8 threads; a CTA holds 4 column slots, the slot being the two
// low lane bits, so that a warp = 4 columns x 8 "j-lanes" (lane = slot + 4*jl) and a column has 2^HB warps (jh).
// The transform is a decimation-in-frequency Cooley-Tukey factorisation N = 8 * 8 * 2^HB whose index bits move between
// registers (3 bits), j-lanes (3 bits) and warps (HB bits):
//
//   load     regs = n[top 3],  jl = n[next 3],  jh = n[HB-1:0]           (rows q*TT + jl*2^HB + jh: natural order in memory)
//   A        radix-8 butterflies in registers, twiddle W_N^(n' r)         -> regs = k1
//   X1       8x8 transpose between registers and j-lanes: warp shuffles, no shared memory, no barrier
//   B        radix-8, twiddle W_(N/8)^(jh r)                              -> regs = k2, jl = k1
//   X2       the ONE shared-memory exchange (CTA barrier): regs <- the next 3 bits of n, j-lanes <- what is left of n
//   C        radix-8 (radix-4 twice when HB = 2)                          -> regs = k3
//   D        HB = 4: twiddle W_16^(n0 r), radix-2 butterfly across lanes 4 apart (shuffle);  HB = 5: W_32^(n r), two of them
//
// The spectrum is left in this digit-permuted order: the pointwise update only needs the frequency index of each
// register (kidx). The inverse runs the transposed flow graph (decimation in time: the same steps in reverse order, the
// same twiddles at the same positions, X2 with its store and load maps swapped) and returns to the row layout of the
// load, so permuted data never reaches memory. inverse = swap re/im, dit, swap re/im (unnormalised).
//
// Shared-memory map of X2 (element index a within a column, physical index a*4 + slot): chosen so that the low bit of a
// differs between the two j-lanes of every quarter warp on both sides of the exchange (a[0] = jl[0] at store XOR jl[0]
// at load), which makes every 16-byte wavefront conflict free, and so that the 8 accesses of a thread are compile-time
// offsets from one base.
#pragma once
#include "fft_core.cuh"

namespace pf {

#if defined(__CUDACC__)
__device__ __forceinline__ double2 shfl_xor_c(double2 v, int m)
{
    return make_double2(__shfl_xor_sync(0xffffffffu, v.x, m), __shfl_xor_sync(0xffffffffu, v.y, m));
}
__device__ __forceinline__ float2 shfl_xor_c(float2 v, int m)
{
    return make_float2(__shfl_xor_sync(0xffffffffu, v.x, m), __shfl_xor_sync(0xffffffffu, v.y, m));
}

// one step of the register <-> lane transpose: register bit BIT is exchanged with lane bit (LANE0 << BIT)
template <int BIT, int LANE0, typename C> __device__ __forceinline__ void transpose_step(C (&v)[8], int lane)
{
    const bool up = (lane & (LANE0 << BIT)) != 0;
#pragma unroll
    for (int q = 0; q < 8; ++q) {
        if (q & (1 << BIT)) continue;
        const int qh = q | (1 << BIT);
        C send = up ? v[q] : v[qh];
        C recv = shfl_xor_c(send, LANE0 << BIT);
        if (up) v[q] = recv; else v[qh] = recv;
    }
}
// v[q] of j-lane jl  <->  v[jl] of j-lane q  (j-lane = (lane / LANE0) & 7)
template <int LANE0, typename C> __device__ __forceinline__ void warp_transpose8(C (&v)[8], int lane)
{
    transpose_step<0, LANE0>(v, lane);
    transpose_step<1, LANE0>(v, lane);
    transpose_step<2, LANE0>(v, lane);
}
// radix-2 butterfly between the lanes MASK apart: the lane whose bit is clear keeps a + b, the other one a - b
template <typename C, typename T> __device__ __forceinline__ void shfl_butterfly(C (&v)[8], int mask, bool up)
{
    const T sgn = up ? T(-1) : T(1);
#pragma unroll
    for (int q = 0; q < 8; ++q) {
        const C p = shfl_xor_c(v[q], mask);
        v[q].x = fma(v[q].x, sgn, p.x);
        v[q].y = fma(v[q].y, sgn, p.y);
    }
}

// v[r] *= w1^r (balanced product tree, as in stage_compute_w)
template <typename C> __device__ __forceinline__ void twiddle_powers(C (&v)[8], C w1)
{
    C w[8];
    w[1] = w1;
#pragma unroll
    for (int r = 2; r < 8; ++r) w[r] = (r & 1) ? cmul(w[r / 2], w[r - r / 2]) : csqr(w[r / 2]);
#pragma unroll
    for (int r = 1; r < 8; ++r) v[r] = cmul(v[r], w[r]);
}
template <int K, typename C> __device__ __forceinline__ void w16_const_all(C (&v)[8])
{
    if constexpr (K < 8) { v[K] = cmul_wconst<16, K>(v[K]); w16_const_all<K + 1>(v); }
}

template <typename T, int N, bool TW_SMEM = false> struct WFft {
    typedef typename V2<T>::type C;
    static constexpr int SLOTS = 4;
    static constexpr int HB = (N == 256) ? 2 : (N == 512) ? 3 : (N == 1024) ? 4 : (N == 2048) ? 5 : -1;
    static_assert(HB >= 2, "warp-tile FFT: N = 256, 512, 1024 or 2048");
    static constexpr int TT = N / 8;
    static constexpr int NW = 1 << HB;              // warps per column = warps per CTA
    static constexpr int THREADS = SLOTS * TT;

    C *buf;                 // N * SLOTS elements of shared memory
    const C *tw;            // exp(-2 pi i k / N): global memory, or shared memory when TW_SMEM
    int lane, sl, jl, jh;
    int sb, lb;             // element bases of the X2 maps (slot included)

    __device__ __forceinline__ WFft(C *smem, const C *twiddles, int tid) : buf(smem), tw(twiddles)
    {
        lane = tid & 31; sl = tid & 3; jl = (tid >> 2) & 7; jh = tid >> 5;
        int s, l;
        if (HB == 2) {
            s = ((jl >> 1) << 6) | (jh << 1) | (jl & 1);
            l = ((jl >> 1) << 6) | (jh << 3) | (jl & 1);
        } else if (HB == 3) {
            s = ((jl >> 1) << 7) | (jh << 1) | (jl & 1);
            l = ((jl >> 1) << 7) | (jh << 4) | (jl & 1);
        } else if (HB == 4) {
            s = ((jl >> 1) << 8) | ((jh >> 1) << 2) | ((jl & 1) << 1) | ((jl & 1) ^ (jh & 1));
            l = ((jl >> 1) << 8) | ((jh >> 1) << 5) | ((jh & 1) << 1) | ((jh & 1) ^ (jl & 1));
        } else {
            s = ((jl >> 2) << 10) | ((jh >> 2) << 4) | (((jl >> 1) & 1) << 3) | (((jh >> 1) & 1) << 2) | ((jl & 1) << 1) | ((jl & 1) ^ (jh & 1));
            l = ((jl >> 2) << 10) | ((jh >> 2) << 7) | (((jh >> 1) & 1) << 3) | (((jl >> 1) & 1) << 2) | ((jh & 1) << 1) | ((jh & 1) ^ (jl & 1));
        }
        sb = s * SLOTS + sl; lb = l * SLOTS + sl;
    }

    // memory row of register q (same before the forward and after the inverse transform)
    __device__ __forceinline__ int row(int q) const { return q * TT + jl * NW + jh; }
    // frequency index of register r after dif()
    __device__ __forceinline__ int kidx(int r) const
    {
        if (HB == 2) return jl + 8 * jh + 32 * (r >> 2) + 64 * (r & 3);
        if (HB == 3) return jl + 8 * jh + 64 * r;
        if (HB == 4) return ((jh & 1) | ((jl >> 1) << 1)) + 8 * (jh >> 1) + 512 * (jl & 1) + 64 * r;
        return ((jh & 3) | ((jl >> 2) << 2)) + 8 * (jh >> 2) + 512 * ((jl >> 1) & 1) + 1024 * (jl & 1) + 64 * r;
    }
    __host__ __device__ static constexpr int soff(int r) { return (r << (HB == 2 ? 3 : HB == 3 ? 4 : HB == 4 ? 5 : 7)) * SLOTS; }
    __host__ __device__ static constexpr int loff(int r)
    {
        return (HB == 2 ? (((r >> 2) << 5) + ((r & 3) << 1)) : (r << (HB == 3 ? 1 : HB == 4 ? 2 : 4))) * SLOTS;
    }

    __device__ __forceinline__ C twv(int i) const { if constexpr (TW_SMEM) return tw[i]; else return __ldg(tw + i); }
    __device__ __forceinline__ C twA() const { return twv(jl * NW + jh); }
    __device__ __forceinline__ C twB() const { return twv(8 * jh); }

    // the shared-memory exchange in two halves, so that a kernel can put work between its barriers
    template <bool FWD> __device__ __forceinline__ void x2_store(const C (&v)[8])
    {
#pragma unroll
        for (int r = 0; r < 8; ++r) buf[(FWD ? sb + soff(r) : lb + loff(r))] = v[r];
    }
    template <bool FWD> __device__ __forceinline__ void x2_load(C (&v)[8]) const
    {
#pragma unroll
        for (int r = 0; r < 8; ++r) v[r] = buf[(FWD ? lb + loff(r) : sb + soff(r))];
    }
    template <bool FWD> __device__ __forceinline__ void x2(C (&v)[8])
    {
        __syncthreads();                          // everyone has taken its elements of the previous exchange
        x2_store<FWD>(v);
        __syncthreads();
        x2_load<FWD>(v);
    }
    __device__ __forceinline__ void last_radix(C (&v)[8])
    {
        if (HB == 2) {                            // radix-4 on register bits 0..1, register bit 2 rides along
            C a[4], b[4];
#pragma unroll
            for (int r = 0; r < 4; ++r) { a[r] = v[r]; b[r] = v[4 + r]; }
            Dft<4>::run(a); Dft<4>::run(b);
#pragma unroll
            for (int r = 0; r < 4; ++r) { v[r] = a[r]; v[4 + r] = b[r]; }
        } else {
            Dft<8>::run(v);
        }
    }

    // forward transform, decimation in frequency: rows row(q) in, frequencies kidx(r) out = dif_a, x2<true>, dif_b
    __device__ __forceinline__ void dif_a(C (&v)[8])
    {
        {
            const C wa = twA();                   // requested before the butterflies that hide its latency
            Dft<8>::run(v);
            twiddle_powers(v, wa);
        }
        {
            const C wb = twB();
            warp_transpose8<SLOTS>(v, lane);
            Dft<8>::run(v);
            twiddle_powers(v, wb);
        }
    }
    __device__ __forceinline__ void dif_b(C (&v)[8])
    {
        last_radix(v);
        if (HB == 4) {
            if (jl & 1) w16_const_all<1>(v);      // W_16^(n0 r)
            shfl_butterfly<C, T>(v, SLOTS, (jl & 1) != 0);
        } else if (HB == 5) {
            twiddle_powers(v, twv(64 * (jl & 3)));                 // W_32^(n[1:0] r)
            shfl_butterfly<C, T>(v, 2 * SLOTS, (jl & 2) != 0);     // over n1
            if ((jl & 3) == 3) {
#pragma unroll
                for (int r = 0; r < 8; ++r) v[r] = cmul_mi(v[r]);  // W_4^(n0 k)
            }
            shfl_butterfly<C, T>(v, SLOTS, (jl & 1) != 0);         // over n0
        }
    }
    __device__ __forceinline__ void dif(C (&v)[8]) { dif_a(v); x2<true>(v); dif_b(v); }

    // the transposed flow graph: frequencies kidx(r) in, rows row(q) out (forward sign, unnormalised) = dit_a, x2<false>, dit_b
    __device__ __forceinline__ void dit_a(C (&v)[8])
    {
        if (HB == 4) {
            shfl_butterfly<C, T>(v, SLOTS, (jl & 1) != 0);
            if (jl & 1) w16_const_all<1>(v);
        } else if (HB == 5) {
            shfl_butterfly<C, T>(v, SLOTS, (jl & 1) != 0);
            if ((jl & 3) == 3) {
#pragma unroll
                for (int r = 0; r < 8; ++r) v[r] = cmul_mi(v[r]);
            }
            shfl_butterfly<C, T>(v, 2 * SLOTS, (jl & 2) != 0);
            twiddle_powers(v, twv(64 * (jl & 3)));
        }
        last_radix(v);
    }
    __device__ __forceinline__ void dit_b(C (&v)[8])
    {
        twiddle_powers(v, twB());
        {
            const C wa = twA();
            Dft<8>::run(v);
            warp_transpose8<SLOTS>(v, lane);
            twiddle_powers(v, wa);
        }
        Dft<8>::run(v);
    }
    __device__ __forceinline__ void dit(C (&v)[8]) { dit_a(v); x2<false>(v); dit_b(v); }
};
#endif

}  // namespace pf
