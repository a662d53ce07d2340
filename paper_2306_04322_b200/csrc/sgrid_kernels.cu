// sgrid_kernels.cu -- small 2D grids: ALL steps of a pf_step_fs(n) call in ONE launch, the state resident in the shared
// memory of a thread-block cluster (SURVEY 8(f)-2 "cluster-resident planes", 8(f)-4 small grids; the paper's remark that
// small grids leave the GPU idle).
//
// A cluster of CS CTAs owns one simulation. CTA r keeps rows [r*RL, (r+1)*RL) (RL = ny/CS) of the z-form of every field
// (row_kernels.cu) and of g = df/dc in its shared memory for the whole call. One step of Algorithm 1:
//   x phase (local rows):   inverse FFT_M of every field in place -> real samples; pointwise g and w_i = eta_i - dt L
//                           df/deta_i (Eq. 13) over the eta_i; forward FFT_M in place         (a6, a1, a2)
//   cluster barrier
//   y phase (mirror pairs of columns, dealt out over all warps of the cluster): a warp gathers its columns from the
//                           slabs of all CTAs through distributed shared memory, unpacks the Hermitian pair, FFT_y,
//                           Eqs. 14-15, inverse FFT_y, repacks and scatters the columns back   (a4, a5)
//   cluster barrier
// Every transform is carried by the lanes of ONE warp (M/8 lanes per row, ny/8 or ny/16 lanes per column), so the FFT
// exchanges need __syncwarp only; the two barriers per step are the only cluster-wide synchronisation, and nothing
// touches global memory between the first and the last step. c^ is carried, as in Algorithm 1: the warp that updates a
// pair of Cahn-Hilliard columns keeps their spectrum in its CTA's shared memory (filled once per launch from the z-form
// of c), so a Cahn-Hilliard column costs two transforms per step like an Allen-Cahn column.
// Square grids 32^2 ... 256^2, both precisions, as far as the state plus the carried c^ fits the shared memory of 16 CTAs:
// every field count up to 128^2 and at 256^2 in fp32; 256^2 in fp64 only with few fields (c + 2 eta no longer fits since c^ is
// carried: sgrid_plan returns 0 and the context stays on the two-kernel path). The host picks the cluster size (1..16).
#include <cooperative_groups.h>

#include "pf_kernels.cuh"
#include "col_buf.cuh"

namespace cg = cooperative_groups;

namespace pf {

namespace {

struct SgWarpSync { __device__ __forceinline__ void operator()() const { __syncwarp(); } };

template <typename C, int LOGPAD> struct SgRowBuf {
    C *base;
    __device__ __forceinline__ void st(int i, C v) { base[i + (i >> LOGPAD)] = v; }
    __device__ __forceinline__ C ld(int i) const { return base[i + (i >> LOGPAD)]; }
    template <int N, int E, int NS> __device__ __forceinline__ void store(const C (&v)[E], int j) { exchange_store<N, E, NS>(v, j, *this); }
    template <int N, int E> __device__ __forceinline__ void load(C (&v)[E], int j) const { exchange_load<N, E>(v, j, *this); }
};

__device__ __forceinline__ double sg_rcp(double x) { return __drcp_rn(x); }
__device__ __forceinline__ float sg_rcp(float x) { return __frcp_rn(x); }
__device__ __forceinline__ double2 sg_shfl1(double2 v)
{
    return make_double2(__shfl_xor_sync(0xffffffffu, v.x, 1), __shfl_xor_sync(0xffffffffu, v.y, 1));
}
__device__ __forceinline__ float2 sg_shfl1(float2 v)
{
    return make_float2(__shfl_xor_sync(0xffffffffu, v.x, 1), __shfl_xor_sync(0xffffffffu, v.y, 1));
}

}  // namespace

template <int M, int NY> struct SgShape {
    static constexpr int EX = 8, TTX = M / EX, UPW = 32 / TTX;            // x transforms: lanes per row, rows per warp pass
    static constexpr int EY = (NY >= 256) ? 16 : 8, TTY = NY / EY;        // y transforms: lanes per column
    static constexpr int SLOTS = 32 / TTY, PWP = SLOTS / 2;               // columns / mirror pairs per warp pass
    static constexpr int LR = (EY >= 16) ? 4 : 3;
    static constexpr int NT = (NY >= 256) ? 256 : 512;
    static constexpr int ROWPITCH = M + (M >> 3) + 1;
    static constexpr int SCR = (UPW * ROWPITCH > NY * SLOTS) ? UPW * ROWPITCH : NY * SLOTS;   // complex elements per warp
    static_assert(TTX >= 2 && TTX <= 32 && TTY >= 2 && TTY <= 16, "transforms must fit a warp");
};

template <typename T, int M, int NY>
__global__ void __launch_bounds__(SgShape<M, NY>::NT, 1) sgrid_kernel(const SgParams<T> p)
{
    typedef typename V2<T>::type C;
    typedef SgShape<M, NY> Sh;
    constexpr int EX = Sh::EX, TTX = Sh::TTX, UPW = Sh::UPW, EY = Sh::EY, TTY = Sh::TTY, SLOTS = Sh::SLOTS, PWP = Sh::PWP;
    constexpr int NT = Sh::NT, NW = NT / 32;
    cg::cluster_group cluster = cg::this_cluster();
    const int CS = (int)cluster.num_blocks();
    const int rank = (int)cluster.block_rank();
    const int rep = blockIdx.x / CS;                       // replica of a batched context
    const int RL = NY / CS;                                // rows of this CTA (a power of two)
    const int rls = __ffs(RL) - 1;
    const int F = p.F;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;

    extern __shared__ __align__(16) unsigned char sg_smem[];
    C *slab = reinterpret_cast<C *>(sg_smem);              // [F + 1][RL][M]; field F = g
    C *s_twm = slab + (size_t)(F + 1) * RL * M;            // exp(-2 pi i k / M)
    C *s_twy = s_twm + M;                                  // exp(-2 pi i k / NY)
    C *s_twx = s_twy + NY;                                 // exp(-2 pi i k / nx), k <= M/2
    C *scratch = s_twx + (M / 2 + 8);                      // [NW][SCR]
    C *carry = scratch + (size_t)NW * Sh::SCR;             // [c tasks of this CTA][EY][32]: c^ of the columns this CTA updates
    const int G = (M / 2 + 1 + PWP - 1) / PWP;             // groups of mirror pairs = Cahn-Hilliard tasks of the cluster
    const int nct = (G + CS - 1) / CS;                     // ... of which this CTA runs at most nct
    T *s_kx2 = reinterpret_cast<T *>(carry + (size_t)nct * EY * 32);      // [M + 1]
    T *s_ky2 = s_kx2 + (M + 1 + 7) / 8 * 8;                // [NY]
    __shared__ C *s_peer[16];                              // the slabs of the cluster's CTAs

    for (int i = tid; i < M; i += NT) s_twm[i] = p.tw_m[i];
    for (int i = tid; i < NY; i += NT) s_twy[i] = p.tw_y[i];
    for (int i = tid; i <= M / 2; i += NT) s_twx[i] = p.twx[i];
    for (int i = tid; i <= M; i += NT) s_kx2[i] = p.kx2[i];
    for (int i = tid; i < NY; i += NT) s_ky2[i] = p.ky2[i];
    if (tid < CS) s_peer[tid] = cluster.map_shared_rank(slab, tid);
    // state -> shared memory
    {
        C *gz = p.zst + (long)rep * NY * M + (long)rank * RL * M;
        for (int f = 0; f < F; ++f)
            for (int i = tid; i < RL * M; i += NT) slab[(long)f * RL * M + i] = gz[(long)f * p.zfs + i];
    }
    cluster.sync();

    C *scr = scratch + (size_t)warp * Sh::SCR;
    const SgWarpSync wsync;
    const T sM = T(1) / T(M), sN = T(1) / T(NY);
    // x transforms: lane -> (row unit of this pass, j)
    const int xu = lane / TTX, xj = lane % TTX;
    SgRowBuf<C, (sizeof(C) == 8 ? 4 : 3)> rbuf{scr + xu * Sh::ROWPITCH};   // one pad element per 128-byte line
    // y transforms: lane -> (column slot, j); slot = pair * 2 + side, the slot is the fastest index
    const int sl = lane % SLOTS, side = sl & 1, yj = lane / SLOTS;
    ColBuf<C, SLOTS, Sh::LR> cbuf{scr, sl};
    const int units = F * RL;                              // (field, local row) transforms of the x phase

    // columns of y-phase task (item, pg): lane -> column slot; returns false for a padding slot
    struct Cols { int colA, colB, col_own, kx; bool store_ok; C wx; T base2; };
    auto task_cols = [&](int pg) {
        Cols k;
        int u = pg * PWP + (sl >> 1);
        const bool valid = u <= M / 2;
        if (!valid) u = 0;
        k.colA = u; k.colB = (M - u) & (M - 1);
        k.kx = side ? M - u : u;
        k.col_own = side ? k.colB : k.colA;
        k.store_ok = valid && (side == 0 || k.colB != k.colA);
        k.wx = s_twx[u];
        k.base2 = s_kx2[k.kx];
        return k;
    };
    // gather the column pair of field fld from the slabs of all CTAs, unpack the Hermitian pair, FFT_y
    auto forward = [&](const Cols &k, int fld, C (&v)[EY]) {
#pragma unroll
        for (int q = 0; q < EY; ++q) {
            const int y = yj + q * TTY;
            const int own = y >> rls;
            const C *src = s_peer[own] + ((long)fld * RL + (y & (RL - 1))) * M;
            const C za = src[k.colA], zb = src[k.colB];
            const C e = mk<T>(T(0.5) * (za.x + zb.x), T(0.5) * (za.y - zb.y));
            const C o = mk<T>(T(0.5) * (za.y + zb.y), T(-0.5) * (za.x - zb.x));
            const C wo = cmul(k.wx, o);
            v[q] = side ? cconj(csub(e, wo)) : cadd(e, wo);
        }
        fft_forward<NY, EY, true>(v, yj, s_twy, cbuf, wsync);
        __syncwarp();
    };
    // c^ of this CTA's Cahn-Hilliard columns from the z-form of c (once per launch; carried in shared memory afterwards,
    // as Algorithm 1 carries it: PAPER.md:176-182 transforms only g and h_i)
    for (int t = rank + CS * warp; t < G; t += CS * NW) {
        const Cols k = task_cols(t);
        C v[EY];
        forward(k, 0, v);
        C *cr = carry + (size_t)(t / CS) * EY * 32 + lane;
#pragma unroll
        for (int q = 0; q < EY; ++q) cr[q * 32] = v[q];
    }
    cluster.sync();

    for (int step = 0; step < p.nsteps; ++step) {
#ifndef PF_SG_SKIP_X
        // ---------------- x phase, pass A: z-form -> real samples, in place ----------------
        for (int g0 = warp * UPW; g0 < units; g0 += NW * UPW) {
            const int u = g0 + xu;
            const bool ok = u < units;
            C *row = slab + (long)(ok ? u : 0) * M;
            C v[EX];
#pragma unroll
            for (int q = 0; q < EX; ++q) v[q] = ok ? cswap(row[xj + q * TTX]) : mk<T>(0, 0);
            fft_forward<M, EX, true>(v, xj, s_twm, rbuf, wsync);
            if (ok) {
#pragma unroll
                for (int q = 0; q < EX; ++q) row[xj + q * TTX] = mk<T>(v[q].y * sM, v[q].x * sM);
            }
            __syncwarp();                                   // the exchange buffer is reused by the next pass
        }
        __syncthreads();
        // ---------------- pass B: g = df/dc, w_i = eta_i - dt L df/deta_i, pointwise ----------------
        for (int i = tid; i < RL * M; i += NT) {
            const C cc = slab[i];
            T h0 = 0, h1 = 0, s0 = 0, s1 = 0;
            for (int f = 1; f < F; ++f) {
                const C e = slab[(long)f * RL * M + i];
                h0 += h_term(e.x); h1 += h_term(e.y);
                s0 += e.x * e.x; s1 += e.y * e.y;
            }
            for (int f = 1; f < F; ++f) {
                const C e = slab[(long)f * RL * M + i];
                slab[(long)f * RL * M + i] = mk<T>(e.x - p.m.dtL * dfdeta(p.m, cc.x, e.x, s0), e.y - p.m.dtL * dfdeta(p.m, cc.y, e.y, s1));
            }
            slab[(long)F * RL * M + i] = mk<T>(dfdc(p.m, cc.x, h0), dfdc(p.m, cc.y, h1));
        }
        __syncthreads();
        // ---------------- pass C: forward FFT_M of every w_i and of g, in place (fields 1 .. F) ----------------
        // (field 0 keeps the dead real samples of c until the y phase writes the new z-form of c over them)
        for (int g0 = warp * UPW; g0 < units; g0 += NW * UPW) {
            const int u = g0 + xu;
            const bool ok = u < units;
            C *row = slab + (long)((ok ? u : 0) + RL) * M;
            C v[EX];
#pragma unroll
            for (int q = 0; q < EX; ++q) v[q] = ok ? row[xj + q * TTX] : mk<T>(0, 0);
            fft_forward<M, EX, true>(v, xj, s_twm, rbuf, wsync);
            if (ok) {
#pragma unroll
                for (int q = 0; q < EX; ++q) row[xj + q * TTX] = v[q];
            }
            __syncwarp();
        }
#endif
        cluster.sync();

        // ---------------- y phase ----------------
#ifndef PF_SG_SKIP_Y
        for (int t = rank + CS * warp; t < F * G; t += CS * NW) {
            const int item = t / G, pg = t - item * G;     // item 0 = c, 1..p = eta_i
            const Cols k = task_cols(pg);
            C v[EY];
            if (item == 0) {
                forward(k, F, v);                           // g^
                // c^ <- (c^ - dt M |xi|^2 g^) / (1 + dt M kappa_c |xi|^4)              Eqs. 12, 14
                C *cr = carry + (size_t)(t / CS) * EY * 32 + lane;
#pragma unroll
                for (int q = 0; q < EY; ++q) {
                    const T k2 = k.base2 + s_ky2[yj + q * TTY];
                    const T d = sg_rcp(T(1) + p.m.dtMkc * k2 * k2);
                    const T a = p.m.dtM * k2;
                    const C cq = cr[q * 32];
                    const C cn = mk<T>((cq.x - a * v[q].x) * d, (cq.y - a * v[q].y) * d);
                    cr[q * 32] = cn;
                    v[q] = cscale(cn, sN);
                }
            } else {
                forward(k, item, v);
                // eta^ <- w^ / (1 + dt L kappa_eta |xi|^2)                             Eqs. 13, 15
#pragma unroll
                for (int q = 0; q < EY; ++q) {
                    const T k2 = k.base2 + s_ky2[yj + q * TTY];
                    v[q] = cscale(v[q], sN * sg_rcp(T(1) + p.m.dtLke * k2));
                }
            }
            // inverse = swap re/im, forward, swap re/im (1/N already applied)
#pragma unroll
            for (int q = 0; q < EY; ++q) v[q] = cswap(v[q]);
            fft_forward<NY, EY, true>(v, yj, s_twy, cbuf, wsync);
            __syncwarp();
            // repack: E = (Ua + conj Ub)/2, W O = (Ua - conj Ub)/2, Z_a = E + i O, Z_b = conj(E - i O)
            const C wxc = cconj(k.wx);
#pragma unroll
            for (int q = 0; q < EY; ++q) {
                const C w = cswap(v[q]);
                const C pv = sg_shfl1(w);
                const C ua = side ? pv : w, ub = side ? w : pv;
                const C e = mk<T>(T(0.5) * (ua.x + ub.x), T(0.5) * (ua.y - ub.y));
                const C wo = mk<T>(T(0.5) * (ua.x - ub.x), T(0.5) * (ua.y + ub.y));
                const C io = cmul_pi(cmul(wxc, wo));
                const C z = side ? cconj(csub(e, io)) : cadd(e, io);
                const int y = yj + q * TTY;
                const int own = y >> rls;
                if (k.store_ok) s_peer[own][((long)item * RL + (y & (RL - 1))) * M + k.col_own] = z;
            }
        }
#endif
        cluster.sync();
    }

    // state -> global memory
    {
        C *gz = p.zst + (long)rep * NY * M + (long)rank * RL * M;
        for (int f = 0; f < F; ++f)
            for (int i = tid; i < RL * M; i += NT) gz[(long)f * p.zfs + i] = slab[(long)f * RL * M + i];
    }
}

template <typename T, int M, int NY> struct SgInst {
    typedef typename V2<T>::type C;
    typedef SgShape<M, NY> Sh;
    static size_t smem(int F, int cs)
    {
        const size_t rl = NY / cs;
        const size_t G = (M / 2 + 1 + Sh::PWP - 1) / Sh::PWP, nct = (G + cs - 1) / cs;
        return sizeof(C) * ((size_t)(F + 1) * rl * M + M + NY + (M / 2 + 8) + (size_t)(Sh::NT / 32) * Sh::SCR + nct * Sh::EY * 32)
             + sizeof(T) * ((size_t)(M + 1 + 7) / 8 * 8 + NY) + 256;
    }
    // smallest cluster size >= want whose slab fits; 0 if none does
    static int plan(int F, int want)
    {
        auto kern = sgrid_kernel<T, M, NY>;
        if (cudaFuncSetAttribute(kern, cudaFuncAttributeNonPortableClusterSizeAllowed, 1) != cudaSuccess) { cudaGetLastError(); }
        for (int cs = want; cs <= 16; cs *= 2) {
            if (cs > NY) break;
            const size_t sm = smem(F, cs);
            if (sm > 227 * 1024) continue;
            if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm) != cudaSuccess) { cudaGetLastError(); continue; }
            cudaLaunchConfig_t cfg = {};
            cfg.gridDim = dim3((unsigned)cs); cfg.blockDim = dim3(Sh::NT); cfg.dynamicSmemBytes = sm;
            cudaLaunchAttribute at[1];
            at[0].id = cudaLaunchAttributeClusterDimension;
            at[0].val.clusterDim.x = (unsigned)cs; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
            cfg.attrs = at; cfg.numAttrs = 1;
            int nclusters = 0;
            if (cudaOccupancyMaxActiveClusters(&nclusters, kern, &cfg) != cudaSuccess) { cudaGetLastError(); continue; }
            if (nclusters >= 1) return cs;
        }
        return 0;
    }
    static cudaError_t launch(const SgParams<T> &p, int cs, int nbatch, cudaStream_t s)
    {
        auto kern = sgrid_kernel<T, M, NY>;
        const size_t sm = smem(p.F, cs);
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm);
        if (e != cudaSuccess) return e;
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3((unsigned)(cs * nbatch)); cfg.blockDim = dim3(Sh::NT); cfg.dynamicSmemBytes = sm; cfg.stream = s;
        cudaLaunchAttribute at[1];
        at[0].id = cudaLaunchAttributeClusterDimension;
        at[0].val.clusterDim.x = (unsigned)cs; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
        cfg.attrs = at; cfg.numAttrs = 1;
        return cudaLaunchKernelEx(&cfg, kern, p);
    }
};

#define PF_SG_DISPATCH(T, nx, ny, CALL)                                      \
    do {                                                                     \
        if (nx == ny) {                                                      \
            switch (nx) {                                                    \
            case 32:  return SgInst<T, 16, 32>::CALL;                        \
            case 64:  return SgInst<T, 32, 64>::CALL;                        \
            case 128: return SgInst<T, 64, 128>::CALL;                       \
            case 256: return SgInst<T, 128, 256>::CALL;                      \
            }                                                                \
        }                                                                    \
    } while (0)

// cluster size for a resident run of an nx x ny grid with F fields (>= want), 0 = shape not served / does not fit
template <typename T> int sgrid_plan(int nx, int ny, int F, int want)
{
    PF_SG_DISPATCH(T, nx, ny, plan(F, want));
    return 0;
}
template <typename T> cudaError_t launch_sgrid(int nx, int ny, const SgParams<T> &p, int cs, int nbatch, cudaStream_t s)
{
    PF_SG_DISPATCH(T, nx, ny, launch(p, cs, nbatch, s));
    return cudaErrorNotSupported;
}

template int sgrid_plan<double>(int, int, int, int);
template int sgrid_plan<float>(int, int, int, int);
template cudaError_t launch_sgrid<double>(int, int, const SgParams<double> &, int, int, cudaStream_t);
template cudaError_t launch_sgrid<float>(int, int, const SgParams<float> &, int, int, cudaStream_t);

}  // namespace pf
