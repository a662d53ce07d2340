// wcol_kernels.cu -- the 2D strided kernel for long fp64 axes (ny = 512, 1024, 2048): SURVEY 8(a) rows a4 + a5 as ONE
// persistent, software-pipelined kernel. Same arithmetic as col_kernel<.., COL_2D_LAST> (col_kernels.cu: Hermitian
// unpack of z-form mirror pairs, FFT_y, spectral update Eqs. 12-15 of PAPER.md:103-116, IFFT_y, repack), different
// execution model:
//
//   * the transform is the warp-tile FFT of wfft.cuh (one shared-memory exchange per transform, shuffles otherwise);
//   * CTAs are persistent (as many as fit the machine) and take work items (field slot, block of two mirror pairs) from
//     an atomic queue, the Cahn-Hilliard items (three transforms) first, so that no CTA idles while items remain;
//   * the z columns of the NEXT pass (the c^ columns after the g^ pass of a Cahn-Hilliard item, the next item otherwise)
//     are fetched with cp.async while the current pass computes: half of them into a landing zone as soon as the
//     current pass has consumed it, the other half into the exchange buffer once its last exchange is over. A pass
//     therefore starts from shared memory and never waits for HBM/L2 latency with nothing else to do (ncu of the
//     non-pipelined kernel: 35 % of all stall samples were long-scoreboard waits on these loads);
//   * the twiddles the transform needs (W_N^i, i < N/8) and the |xi_y|^2 table live in shared memory.
//
// Shared memory per CTA (N = 1024): exchange buffer 64 KB + landing zone 32 KB + tables 10 KB = 106 KB, two CTAs per SM.
#include "pf_kernels.cuh"
#include "wfft.cuh"

namespace pf {

namespace {

__device__ __forceinline__ double rcpw(double x) { return __drcp_rn(x); }

__device__ __forceinline__ void cp_async16(void *smem_dst, const void *gmem_src)
{
    const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(d), "l"(gmem_src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }

}  // namespace

template <typename T, int N>
__global__ void __launch_bounds__(WFft<T, N>::THREADS, (WFft<T, N>::THREADS >= 1024) ? 1 : (1024 / WFft<T, N>::THREADS > 4 ? 4 : 1024 / WFft<T, N>::THREADS))
wcol2d_kernel(const ColParams<T> p, const int nblk, const int nitems)
{
    typedef typename V2<T>::type C;
    typedef WFft<T, N, true> W;
    constexpr int GT = W::THREADS, TT = W::TT, E = 8, TP = 2;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    C *X = reinterpret_cast<C *>(smem_raw);                 // N * 4 elements: exchange buffer; landing zone of rows q >= 4
    C *L = X + (size_t)N * 4;                               // 4 * GT elements: landing zone of rows q < 4
    C *s_tw = L + 4 * GT;                                   // TT twiddles
    T *s_k2 = reinterpret_cast<T *>(s_tw + TT);             // N frequencies
    int *s_item = reinterpret_cast<int *>(s_k2 + N);

    const int tid = threadIdx.x;
    const int side = tid & 1;
    const int M = p.M;
    W wf(X, s_tw, tid);

    for (int i = tid; i < TT; i += GT) s_tw[i] = p.tw[i];
    for (int i = tid; i < N; i += GT) s_k2[i] = p.ky2[i];
    if (tid == 0) s_item[0] = atomicAdd(p.queue, 1);
    __syncthreads();
    int it = s_item[0];

    // ---- per-item state ----
    int slot, ub, zcolA, zcolB, kx;
    bool store_ok, is_c;
    T base2;
    C wx;
    auto decode = [&](int id) {
        slot = id / nblk; ub = id - slot * nblk;
        int u = ub * TP + ((tid & 3) >> 1);
        const bool valid = (u <= M / 2);
        if (!valid) u = 0;
        zcolA = u; zcolB = (M - u) & (M - 1);
        kx = side ? M - u : u;
        store_ok = valid && (side == 0 || zcolB != zcolA);
        wx = p.twx[u];
        base2 = p.kx2[kx];
        is_c = p.has_c && slot == 0;
    };
    // source array of a pass: the g pass of a Cahn-Hilliard item reads in1, everything else the state of its slot
    auto src_of = [&](int sl_, bool gpass) -> const C * { return gpass ? p.in1 : p.in0 + (long)sl_ * p.in_fs; };
    // cp.async of this thread's own z column, rows q in [Q0, Q1): rows q < 4 land in L, the others in X
    auto fetch_rows = [&](const C *src, int col, int q0, int q1) {
#pragma unroll
        for (int q = 0; q < E; ++q) {
            if (q < q0 || q >= q1) continue;
            C *dst = (q < 4) ? (L + q * GT + tid) : (X + (q - 4) * GT + tid);
            cp_async16(dst, src + (long)wf.row(q) * p.in_rs + col);
        }
        cp_async_commit();
    };

    grid_dependency_wait();                // everything above touches constant tables and the queue only
    grid_dependents_launch();
    if (it >= nitems) goto finish;
    decode(it);
    {
        bool gpass = is_c;
        fetch_rows(src_of(slot, gpass), side ? zcolB : zcolA, 0, 8);

        C v[E];
        while (true) {
            // ---- the z columns of this pass have landed (own copies: wait_group; the partner's: same warp) ----
            cp_async_wait_all();
            __syncwarp();
#pragma unroll
            for (int q = 0; q < E; ++q) {
                const C *land = (q < 4) ? (L + q * GT) : (X + (q - 4) * GT);
                const C za = land[tid & ~1], zb = land[tid | 1];
                // E = (za + conj zb)/2, O = -(i/2)(za - conj zb), U_u = E + W O, U_{M-u} = conj(E - W O)
                const C e = mk<T>(T(0.5) * (za.x + zb.x), T(0.5) * (za.y - zb.y));
                const C o = mk<T>(T(0.5) * (za.y + zb.y), T(-0.5) * (za.x - zb.x));
                const C wo = cmul(wx, o);
                v[q] = side ? cconj(csub(e, wo)) : cadd(e, wo);
            }
            if (!gpass && tid == 0) s_item[1] = atomicAdd(p.queue, 1);       // the item after this one
            wf.dif_a(v);
            __syncthreads();               // B1: everyone has consumed L and X; s_item[1] is visible
            // ---- what the next pass reads: rows q < 4 now (L is free), rows q >= 4 after the last exchange ----
            const int nit = gpass ? it : s_item[1];
            const bool more = gpass || nit < nitems;
            int ncol = side ? zcolB : zcolA;
            const C *nsrc = nullptr;
            if (more) {
                if (gpass) nsrc = src_of(slot, false);
                else {
                    const int nslot = nit / nblk, nub = nit - nslot * nblk;
                    int u = nub * TP + ((tid & 3) >> 1);
                    if (u > M / 2) u = 0;
                    ncol = side ? ((M - u) & (M - 1)) : u;
                    nsrc = src_of(nslot, p.has_c && nslot == 0);
                }
                fetch_rows(nsrc, ncol, 0, 4);
            }
            wf.template x2_store<true>(v);
            __syncthreads();
            wf.template x2_load<true>(v);
            wf.dif_b(v);

            C *park = p.park + ((long)ub * E) * GT + tid;
            if (gpass) {
                // Cahn-Hilliard, first transform: dt M |xi|^2 g^ parked in global memory (thread-linear, stays in L2)
#pragma unroll
                for (int q = 0; q < E; ++q) park[(long)q * GT] = cscale(v[q], p.m.dtM * (base2 + s_k2[wf.kidx(q)]));
                __syncthreads();           // B3: the exchange buffer is free
                fetch_rows(nsrc, ncol, 4, 8);
                gpass = false;
                continue;
            }

            // ---- spectral update (1/N folded in), Eqs. 14-15 ----
            const T s = T(1) / T(N);
            if (is_c) {
#pragma unroll
                for (int q = 0; q < E; ++q) {
                    const T k2 = base2 + s_k2[wf.kidx(q)];
                    const T d = s * rcpw(T(1) + p.m.dtMkc * k2 * k2);
                    const C gq = park[(long)q * GT];
                    v[q] = mk<T>((v[q].x - gq.x) * d, (v[q].y - gq.y) * d);
                }
            } else {
#pragma unroll
                for (int q = 0; q < E; ++q) {
                    const T k2 = base2 + s_k2[wf.kidx(q)];
                    v[q] = cscale(v[q], s * rcpw(T(1) + p.m.dtLke * k2));
                }
            }
            // ---- inverse = swap re/im, transposed flow graph, swap re/im ----
#pragma unroll
            for (int q = 0; q < E; ++q) v[q] = cswap(v[q]);
            wf.dit_a(v);
            __syncthreads();
            wf.template x2_store<false>(v);
            __syncthreads();
            wf.template x2_load<false>(v);
            __syncthreads();               // B3: the exchange buffer is free
            if (more) fetch_rows(nsrc, ncol, 4, 8);
            wf.dit_b(v);
            // ---- repack: E = (Ua + conj Ub)/2, W O = (Ua - conj Ub)/2, Z_a = E + i O, Z_b = conj(E - i O) ----
            {
                const C wxc = cconj(wx);
                C *dst = p.out + (long)slot * p.out_fs + (side ? zcolB : zcolA);
#pragma unroll
                for (int q = 0; q < E; ++q) {
                    const C mine = mk<T>(v[q].y, v[q].x);
                    const C pv = shfl_xor_c(mine, 1);
                    const C ua = side ? pv : mine, ubv = side ? mine : pv;
                    const C e = mk<T>(T(0.5) * (ua.x + ubv.x), T(0.5) * (ua.y - ubv.y));
                    const C wo = mk<T>(T(0.5) * (ua.x - ubv.x), T(0.5) * (ua.y + ubv.y));
                    const C io = cmul_pi(cmul(wxc, wo));
                    const C z = side ? cconj(csub(e, io)) : cadd(e, io);
                    if (store_ok) dst[(long)wf.row(q) * p.out_rs] = z;
                }
            }
            if (!more) break;
            it = nit;
            decode(it);
            gpass = is_c;
        }
    }
finish:
    // the last CTA to leave re-arms the queue for the next launch
    __syncthreads();
    if (tid == 0) {
        __threadfence();
        if (atomicAdd(p.queue + 1, 1) == (int)gridDim.x - 1) { p.queue[0] = 0; p.queue[1] = 0; __threadfence(); }
    }
}

template <typename T, int N> static cudaError_t launch_wcol2d_inst(int nslots, const ColParams<T> &p, cudaStream_t s)
{
    typedef typename V2<T>::type C;
    typedef WFft<T, N> W;
    const int nblk = (p.M / 2 + 2) / 2;                    // blocks of two mirror pairs (u = 0 .. M/2)
    const int nitems = nblk * nslots;
    const size_t smem = (size_t)N * 4 * sizeof(C) + (size_t)4 * W::THREADS * sizeof(C) + (size_t)W::TT * sizeof(C) +
                        (size_t)N * sizeof(T) + 16;
    auto kern = wcol2d_kernel<T, N>;
    // attribute and occupancy per launch: both are per device, and this opt-in variant is no hot path
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    int dev = 0, sms = 0, per_sm = 0;
    if ((e = cudaGetDevice(&dev)) != cudaSuccess) return e;
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, W::THREADS, smem);
    if (e != cudaSuccess) return e;
    if (per_sm < 1) return cudaErrorLaunchOutOfResources;
    const int max_ctas = sms * per_sm;
    const int grid = nitems < max_ctas ? nitems : max_ctas;
    return launch_pdl(kern, dim3((unsigned)grid), dim3(W::THREADS), smem, s, p.pdl != 0, p, nblk, nitems);
}

// ny = 512, 1024, 2048 in fp64; returns cudaErrorNotSupported for everything else (the caller then uses col_kernel)
template <typename T> cudaError_t launch_wcol2d(int nfft, int nslots, const ColParams<T> &p, cudaStream_t s)
{
    if constexpr (sizeof(T) == 8) {
        switch (nfft) {
        case 512:  return launch_wcol2d_inst<T, 512>(nslots, p, s);
        case 1024: return launch_wcol2d_inst<T, 1024>(nslots, p, s);
        case 2048: return launch_wcol2d_inst<T, 2048>(nslots, p, s);
        }
    }
    return cudaErrorNotSupported;
}

template cudaError_t launch_wcol2d<double>(int, int, const ColParams<double> &, cudaStream_t);
template cudaError_t launch_wcol2d<float>(int, int, const ColParams<float> &, cudaStream_t);

}  // namespace pf
