// col2d_kernels.cu -- the 2D last-axis kernel of the Fourier-spectral step (SURVEY 8(a) rows a4 + a5): forward FFT_y,
// spectral update (Eqs. 12-15), inverse FFT_y, on the z-form state of row_kernels.cu.
//
// Same transform, thread layout and exchange buffer as col_kernels.cu (one column per thread group, mirror pairs
// (u, M-u) of the z-form unpacked to the true half-spectrum columns before the transform and repacked after the
// inverse). Two things differ:
//
//  * c^ is CARRIED between steps, as the paper does (Alg. 1: only g, h_i are transformed; c^(t) is
//    kept): the full 2D spectrum of c lives in `carry`, in the thread-linear order of this kernel (thread tid of the CTA
//    that owns column block ub keeps its E values at carry[(ub*E + q)*THREADS + tid], so every access is a contiguous
//    16-byte-per-lane stream). A Cahn-Hilliard block therefore costs TWO transforms (FFT_y g, IFFT_y c^') like an
//    Allen-Cahn block, not three, and dt M |xi|^2 g^ never has to be parked.
//  * the work is a STATIC, BALANCED SCHEDULE instead of one CTA per (field, block): the host deals transform passes
//    ("rounds") to as many CTAs as are resident at once so that every CTA gets the same number. A Cahn-Hilliard block is
//    two one-round items, C_FWD (g^ -> update -> carry) and C_INV (carry -> IFFT -> z-form), which may run in different
//    CTAs (a flag in global memory orders them; the producer never waits, consumers start after their producers, so
//    there is no deadlock however few CTAs are resident); an Allen-Cahn block is one two-round item. 1024^2, c + 2 eta:
//    129 blocks x 6 rounds = 774 rounds = 258 CTAs x 3 rounds -- one wave, no tail (the one-CTA-per-item form was 387
//    CTAs of 3 or 2 rounds on 296 slots: 30 % of the SM cycles idle, profiles/r1_ncu_full_1024sq.md).
#include <algorithm>
#include <queue>
#include <vector>

#include "pf_kernels.cuh"
#include "col_buf.cuh"

#ifndef PF_COL2D_TP2048
#define PF_COL2D_TP2048 2
#endif

namespace pf {

namespace {

__device__ __forceinline__ double rcp2(double x) { return __drcp_rn(x); }
__device__ __forceinline__ float rcp2(float x) { return __frcp_rn(x); }
__device__ __forceinline__ double2 shfl1(double2 v)
{
    return make_double2(__shfl_xor_sync(0xffffffffu, v.x, 1), __shfl_xor_sync(0xffffffffu, v.y, 1));
}
__device__ __forceinline__ float2 shfl1(float2 v)
{
    return make_float2(__shfl_xor_sync(0xffffffffu, v.x, 1), __shfl_xor_sync(0xffffffffu, v.y, 1));
}
__device__ __forceinline__ double2 ld_cg(const double2 *p) { return __ldcg(p); }
__device__ __forceinline__ float2 ld_cg(const float2 *p) { return __ldcg(p); }
__device__ __forceinline__ void st_cg(double2 *p, double2 v) { __stcg(p, v); }
__device__ __forceinline__ void st_cg(float2 *p, float2 v) { __stcg(p, v); }
__device__ __forceinline__ void prefetch_l2(const void *p) { asm volatile("prefetch.global.L2 [%0];" ::"l"(p)); }
__device__ __forceinline__ int ld_acquire(const int *p)
{
    int v;
    asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_release(int *p, int v) { asm volatile("st.release.gpu.global.s32 [%0], %1;" ::"l"(p), "r"(v) : "memory"); }

struct CtaSync2 { __device__ __forceinline__ void operator()() const { __syncthreads(); } };

template <int N, int E, int TP> struct Col2dShape {
    static constexpr int TT = N / E;
    static constexpr int SLOTS = 2 * TP;
    static constexpr int THREADS = SLOTS * TT;
    static constexpr int MINB = (THREADS >= 1024) ? 1 : ((1024 / THREADS > 32) ? 32 : 1024 / THREADS);
    static constexpr int LR = (E >= 16) ? 4 : 3;
    static constexpr int MAXITEMS = 32;                                   // items of a place kept in shared memory
};

}  // namespace

// L2 prefetch of the slice of the carried spectrum a Cahn-Hilliard item reads, one lane per 128-byte line
template <typename T, int E, int GT>
__device__ __forceinline__ void prefetch_carry(const Col2dParams<T> &p, int item, int tid)
{
    typedef typename V2<T>::type C;
    const int op = item & 15, ub = item >> 8;
    if ((op == COL2D_C_FWD || op == COL2D_C_FULL) && (tid & (128 / (int)sizeof(C) - 1)) == 0) {
        const C *carry = p.carry + ((long)ub * E) * GT + tid;
#pragma unroll
        for (int q = 0; q < E; ++q) prefetch_l2(carry + (long)q * GT);
    }
}

template <typename T, int N, int E, int TP>
__global__ void __launch_bounds__(Col2dShape<N, E, TP>::THREADS, Col2dShape<N, E, TP>::MINB)
col2d_kernel(const Col2dParams<T> p)
{
    typedef typename V2<T>::type C;
    typedef Col2dShape<N, E, TP> Sh;
    constexpr int TT = Sh::TT, SLOTS = Sh::SLOTS, GT = Sh::THREADS;
    static_assert(GT % 32 == 0, "a CTA must be whole warps");

#ifdef PF_TRACE
    TraceScope trace(p.trace, 1);
#endif
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ int s_items[Sh::MAXITEMS];
    const int tid = threadIdx.x;
    const int sl = tid % SLOTS;                        // column slot: side = sl & 1, pair = sl >> 1
    const int side = sl & 1;
    const int j = tid / SLOTS;
    const int M = p.M;
    ColBuf<C, SLOTS, Sh::LR> buf{reinterpret_cast<C *>(smem_raw), sl};
    // |xi_y|^2 of the FFT axis behind the exchange buffer: eight scattered 8-byte reads per update and thread otherwise
    T *s_k2 = reinterpret_cast<T *>(reinterpret_cast<C *>(smem_raw) + (size_t)N * SLOTS);
    // (the twiddle table in shared memory as well was measured slower: 88 KB per CTA needs the next carve-out)
    const CtaSync2 sync;

    // Place in the schedule = a ticket, taken in the order in which CTAs START (not blockIdx: CUDA promises neither that
    // CTAs are dispatched in index order nor that the whole grid is resident at once, e.g. when a second context keeps SMs
    // busy). Every place lists its C_FWD items -- which wait for nothing -- first, and the consumer of a block sits at a
    // place >= its producer's; a place is only ever held by a CTA that is already running, so a waiting consumer's
    // producer is on the machine and finishes: forward progress does not depend on the scheduler.
    // The counter wraps to zero with the grid's last ticket (atomicInc). It is taken BEFORE griddepcontrol.launch_dependents:
    // the next launch of this kernel sits two programmatic edges downstream, so none of its CTAs exists before every CTA of
    // this launch has its ticket. p.ticket == nullptr (PF_COL2D_NOTICKET=1, A/B runs): place = blockIdx.x.
    __shared__ int s_place;
    for (int i = tid; i < N; i += GT) s_k2[i] = p.ky2[i];
    if (tid == 0) s_place = p.ticket ? (int)atomicInc(p.ticket, gridDim.x - 1) : (int)blockIdx.x;
    __syncthreads();
    const int place = s_place;

    grid_dependency_wait();                // everything above touches constant tables and the ticket only
    grid_dependents_launch();

    const T sN = T(1) / T(N);
    for (int it = 0; it < p.per_cta; ++it) {
        const int ic = it % Sh::MAXITEMS;
        if (ic == 0) {                             // the next MAXITEMS items of this place
            __syncthreads();
            if (tid < Sh::MAXITEMS) s_items[tid] = (it + tid < p.per_cta) ? p.sched[(long)place * p.per_cta + it + tid] : -1;
            __syncthreads();
        }
        const int item = s_items[ic];
        if (item < 0) break;
        // block index over all replicas of a batched context (pf_create_batch): gb = replica * nblk + block
        const int op = item & 15, slot = (item >> 4) & 15, gb = item >> 8;
        const int rep = gb / p.nblk, ub = gb - rep * p.nblk;

        // ---- the columns of this item ----
        int u = ub * TP + (sl >> 1);
        const bool valid = (u <= M / 2);
        if (!valid) u = 0;
        const int zcolA = u, zcolB = (M - u) & (M - 1);
        const int kx = side ? M - u : u;
        const bool store_ok = valid && (side == 0 || zcolB != zcolA);
        const C wx = p.twx[u];                     // exp(-2 pi i u / nx)
        const T base2 = p.kx2[kx];
        C *carry = p.carry + ((long)gb * E) * GT + tid;
        const long rep_off = (long)rep * N * M;            // rows of this replica within a field
        C *zfield = p.zst + (long)slot * p.zfs + rep_off;

        // the carried spectrum was written a step ago: ask the L2 for this item's slice (first item) and the next item's
        if (ic == 0) prefetch_carry<T, E, GT>(p, item, tid);
        if (ic + 1 < Sh::MAXITEMS && s_items[ic + 1] >= 0) prefetch_carry<T, E, GT>(p, s_items[ic + 1], tid);

        C v[E];
        if (op != COL2D_C_INV) {
            // E = (za + conj zb)/2, O = -(i/2)(za - conj zb), U_u = E + W O (side 0), U_{M-u} = conj(E - W O) (side 1)
            const C *src = (op == COL2D_C_FWD || op == COL2D_C_FULL) ? p.zg + rep_off : zfield;
#pragma unroll
            for (int q = 0; q < E; ++q) {
                const long i = j + q * TT;
                const C za = src[i * M + zcolA], zb = src[i * M + zcolB];
                const C e = mk<T>(T(0.5) * (za.x + zb.x), T(0.5) * (za.y - zb.y));
                const C o = mk<T>(T(0.5) * (za.y + zb.y), T(-0.5) * (za.x - zb.x));
                const C wo = cmul(wx, o);
                v[q] = side ? cconj(csub(e, wo)) : cadd(e, wo);
            }
            fft_forward<N, E>(v, j, p.tw, buf, sync);
        }

        if (op == COL2D_ETA) {
            // eta^ <- w^ / (1 + dt L kappa_eta |xi|^2)                                    Eqs. 13, 15
#pragma unroll
            for (int q = 0; q < E; ++q) {
                const T k2 = base2 + s_k2[j + q * TT];
                v[q] = cscale(v[q], sN * rcp2(T(1) + p.m.dtLke * k2));
            }
        } else if (op == COL2D_C_INIT) {
            // pf_set_fields: the carried spectrum is FFT_y of the unpacked z-form of c
#pragma unroll
            for (int q = 0; q < E; ++q) st_cg(carry + (long)q * GT, v[q]);
            continue;
        } else if (op == COL2D_C_FWD || op == COL2D_C_FULL) {
            // c^ <- (c^ - dt M |xi|^2 g^) / (1 + dt M kappa_c |xi|^4)                      Eqs. 12, 14
#pragma unroll
            for (int q = 0; q < E; ++q) {
                const T k2 = base2 + s_k2[j + q * TT];
                const T d = rcp2(T(1) + p.m.dtMkc * k2 * k2);
                const T a = p.m.dtM * k2;
                const C cq = ld_cg(carry + (long)q * GT);
                v[q] = mk<T>((cq.x - a * v[q].x) * d, (cq.y - a * v[q].y) * d);
                st_cg(carry + (long)q * GT, v[q]);
            }
            if (op == COL2D_C_FWD) {
                __syncthreads();                               // the carry writes of the whole CTA precede the flag
                if (tid == 0) { __threadfence(); st_release(p.flags + gb, 1); }
                continue;
            }
#pragma unroll
            for (int q = 0; q < E; ++q) v[q] = cscale(v[q], sN);
        } else {   // COL2D_C_INV
            if (tid == 0) {
                while (ld_acquire(p.flags + gb) == 0) __nanosleep(100);
                p.flags[gb] = 0;                   // one producer and one consumer per launch
            }
            __syncthreads();
#pragma unroll
            for (int q = 0; q < E; ++q) v[q] = cscale(ld_cg(carry + (long)q * GT), sN);
        }

        // inverse = swap re/im, forward, swap re/im (1/N already applied)
#pragma unroll
        for (int q = 0; q < E; ++q) v[q] = cswap(v[q]);
        fft_forward<N, E>(v, j, p.tw, buf, sync);
#pragma unroll
        for (int q = 0; q < E; ++q) v[q] = cswap(v[q]);

        // E = (Ua + conj Ub)/2, W O = (Ua - conj Ub)/2, Z_a = E + i O, Z_b = conj(E - i O); partner = neighbouring lane
        const C wxc = cconj(wx);
        C *dst = zfield + (side ? zcolB : zcolA);
#pragma unroll
        for (int q = 0; q < E; ++q) {
            const C pv = shfl1(v[q]);
            const C ua = side ? pv : v[q], ubv = side ? v[q] : pv;
            const C e = mk<T>(T(0.5) * (ua.x + ubv.x), T(0.5) * (ua.y - ubv.y));
            const C wo = mk<T>(T(0.5) * (ua.x - ubv.x), T(0.5) * (ua.y + ubv.y));
            const C io = cmul_pi(cmul(wxc, wo));
            const C z = side ? cconj(csub(e, io)) : cadd(e, io);
            if (store_ok) dst[(long)(j + q * TT) * M] = z;
        }
    }

#ifdef PF_TRACE
    trace.finish();
#endif
}

// ---------------------------------------------------------------- host: schedule + launch ----------
template <typename T, int N, int E, int TP> struct Col2dInst {
    typedef typename V2<T>::type C;
    typedef Col2dShape<N, E, TP> Sh;
        static size_t smem() { return (size_t)N * Sh::SLOTS * sizeof(C) + (size_t)N * sizeof(T); }
    // shared memory of the CTAs that share an SM (1 KB per CTA is the system's), as a percentage of the 228 KB maximum
    static int carveout()
    {
        const size_t per_cta = smem() + 1024 + 256;
        size_t per_sm = (size_t)Sh::MINB * per_cta;
        if (per_sm > 228 * 1024) per_sm = (228 * 1024 / per_cta) * per_cta;
        int pct = (int)((per_sm * 100 + 228 * 1024 - 1) / (228 * 1024));
        return pct > 100 ? 100 : pct;
    }
    static cudaError_t prepare()
    {
        auto kern = col2d_kernel<T, N, E, TP>;
        cudaError_t e = cudaSuccess;
        if (smem() > 48 * 1024) e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem());
        if (e == cudaSuccess) e = cudaFuncSetAttribute(kern, cudaFuncAttributePreferredSharedMemoryCarveout, carveout());
        return e;
    }
    static cudaError_t shape(int M, Col2dShapeInfo *o)
    {
        cudaError_t e = prepare();
        if (e != cudaSuccess) return e;
        int dev = 0, sms = 0, per_sm = 0;
        if ((e = cudaGetDevice(&dev)) != cudaSuccess) return e;
        if ((e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess) return e;
        if ((e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, col2d_kernel<T, N, E, TP>, Sh::THREADS, smem())) != cudaSuccess) return e;
        o->tp = TP; o->e = E; o->threads = Sh::THREADS; o->max_items = Sh::MAXITEMS;
        o->nblk = (M / 2 + TP) / TP;
        o->slots = sms * (per_sm > 0 ? per_sm : 1);               // places in the schedule = resident CTAs
        o->carry_elems = (long)o->nblk * E * Sh::THREADS;
        o->carveout_pct = carveout();
        return cudaSuccess;
    }
    static cudaError_t launch(const Col2dParams<T> &p, int grid, cudaStream_t s)
    {
        cudaError_t e = prepare();
        if (e != cudaSuccess) return e;
        return launch_pdl(col2d_kernel<T, N, E, TP>, dim3((unsigned)grid), dim3(Sh::THREADS), smem(), s, p.pdl != 0, p);
    }
};

// column pairs per CTA: whole warps at short axes, 32-byte (fp64) / 32..64-byte (fp32) global pieces at long ones (the
// shapes col_kernels.cu was tuned to on B200)
#define PF_COL2D_DISPATCH(T, nfft, CALL)                                         \
    do {                                                                         \
        if constexpr (sizeof(T) == 4) {                                          \
            if (nfft == 1024) return Col2dInst<T, 1024, 16, 4>::CALL;            \
            if (nfft == 2048) return Col2dInst<T, 2048, 16, 2>::CALL;            \
        } else {                                                                 \
            if (nfft == 1024) return Col2dInst<T, 1024, 8, 2>::CALL;             \
            if (nfft == 2048) return Col2dInst<T, 2048, 8, PF_COL2D_TP2048>::CALL; \
        }                                                                        \
        switch (nfft) {                                                          \
        case 16:   return Col2dInst<T, 16, 8, 8>::CALL;                          \
        case 32:   return Col2dInst<T, 32, 8, 8>::CALL;                          \
        case 64:   return Col2dInst<T, 64, 8, 4>::CALL;                          \
        case 128:  return Col2dInst<T, 128, 8, 4>::CALL;                         \
        case 256:  return Col2dInst<T, 256, 8, 4>::CALL;                         \
        case 512:  return Col2dInst<T, 512, 8, 2>::CALL;                         \
        }                                                                        \
        return cudaErrorInvalidValue;                                            \
    } while (0)

template <typename T> cudaError_t col2d_shape(int nfft, int M, Col2dShapeInfo *o) { PF_COL2D_DISPATCH(T, nfft, shape(M, o)); }
template <typename T> cudaError_t launch_col2d(int nfft, const Col2dParams<T> &p, int grid, cudaStream_t s) { PF_COL2D_DISPATCH(T, nfft, launch(p, grid, s)); }

template cudaError_t col2d_shape<double>(int, int, Col2dShapeInfo *);
template cudaError_t col2d_shape<float>(int, int, Col2dShapeInfo *);
template cudaError_t launch_col2d<double>(int, const Col2dParams<double> &, int, cudaStream_t);
template cudaError_t launch_col2d<float>(int, const Col2dParams<float> &, int, cudaStream_t);

// Deals the items of one step to CTAs (see the header comment). Rounds: C_FWD 1, C_INV 1, ETA 2. Every CTA lists its
// C_FWD items first and its C_INV items last; the consumer of block b sits in a CTA whose index is >= its producer's.
// A C_INV that directly follows its own C_FWD in the same CTA is merged into C_FULL (values stay in registers).
void col2d_schedule(int nblk, int n_eta, int slots, int *grid_out, int *per_cta_out, std::vector<int> &sched)
{
    const long total = (long)nblk * (2 + 2 * n_eta);
    long rmax = (total + slots - 1) / slots;
    if (rmax < 2) rmax = 2;
    int G = (int)((total + rmax - 1) / rmax);
    if (G < 1) G = 1;
    if (G > slots) G = slots;
    std::vector<std::vector<int>> list(G);
    std::vector<int> load(G, 0), prod(nblk, 0);
    auto enc = [](int op, int slot, int b) { return op | (slot << 4) | (b << 8); };
    for (int b = 0; b < nblk; ++b) { const int c = b % G; prod[b] = c; list[c].push_back(enc(COL2D_C_FWD, 0, b)); load[c] += 1; }
    typedef std::pair<int, int> LI;                                   // (load, cta): least loaded, then lowest index
    std::priority_queue<LI, std::vector<LI>, std::greater<LI>> pq;
    for (int c = 0; c < G; ++c) pq.push(LI(load[c], c));
    for (int b = 0; b < nblk; ++b)
        for (int s = 1; s <= n_eta; ++s) {
            const LI t = pq.top(); pq.pop();
            list[t.second].push_back(enc(COL2D_ETA, s, b));
            load[t.second] += 2;
            pq.push(LI(load[t.second], t.second));
        }
    for (int b = 0; b < nblk; ++b) {
        int best = prod[b];
        for (int c = prod[b]; c < G; ++c) if (load[c] < load[best]) best = c;
        if (best == prod[b] && list[best].back() == enc(COL2D_C_FWD, 0, b)) list[best].back() = enc(COL2D_C_FULL, 0, b);
        else list[best].push_back(enc(COL2D_C_INV, 0, b));
        load[best] += 1;
    }
    size_t per = 1;
    for (auto &l : list) per = std::max(per, l.size());
    sched.assign((size_t)G * per, -1);
    for (int c = 0; c < G; ++c) std::copy(list[c].begin(), list[c].end(), sched.begin() + (size_t)c * per);
    *grid_out = G; *per_cta_out = (int)per;
}

// items of the one-off pass that fills `carry` from the z-form of c (after pf_set_fields / an FD step)
void col2d_schedule_init(int nblk, int slots, int *grid_out, int *per_cta_out, std::vector<int> &sched)
{
    const int G = std::min(nblk, slots);
    const int per = (nblk + G - 1) / G;
    sched.assign((size_t)G * per, -1);
    for (int b = 0; b < nblk; ++b) sched[(size_t)(b % G) * per + b / G] = COL2D_C_INIT | (b << 8);
    *grid_out = G; *per_cta_out = per;
}

}  // namespace pf
