// fd2d_kernels.cu -- the explicit forward-Euler finite-difference step in 2D, 5-point
// Laplacian, periodic wrap, every right-hand side at time t, ONE launch per step, pair-wide form of fd_fused2d_kernel
// (fd_kernels.cu) for nx >= 64, ny >= 16:
//     mu = df/dc - kappa_c lap c,   c' = c + dt M lap mu,   eta_i' = eta_i - dt L (df/deta_i - kappa_eta lap eta_i).
// A CTA stages a 64 x 16 tile in shared memory -- c with a halo of two points, every eta_i with a halo of one (two in x, so that
// every copy is an aligned pair) -- forms mu on the tile plus a ring of one point, then the new c and eta_i. Every thread owns TWO
// neighbouring x points in each of two rows: shared-memory reads, cp.async tile loads and global stores move 16-byte pairs (fp64),
// and the centre values of a thread's own points stay in registers between the two phases. The ring of mu is dealt out warp by
// warp (two extra rows: warps 0 and 1; two extra columns: warps 2 and 3), as in fd3d_kernels.cu.
#include "pf_kernels.cuh"

namespace pf {

namespace {

template <typename T> struct Pair2;
template <> struct Pair2<double> { typedef double2 type; };
template <> struct Pair2<float>  { typedef float2  type; };

template <typename T> __device__ __forceinline__ void cp_async_pair2(T *smem_dst, const T *gmem_src)
{
    asm volatile("cp.async.ca.shared.global [%0], [%1], %2;" ::"r"((unsigned)__cvta_generic_to_shared(smem_dst)), "l"(gmem_src), "n"(2 * sizeof(T)) : "memory");
}

}  // namespace

template <typename T, int NE>
__global__ void __launch_bounds__(256) fd2d_pair_kernel(const FdParams<T> p)
{
    typedef typename Pair2<T>::type P2;
    constexpr int TX = 64, TY = 16, PW = TX + 4;
    constexpr int CH = TY + 4, EH = TY + 2, CP = CH * PW, EP = EH * PW;
    extern __shared__ __align__(16) unsigned char fd2_smem[];
    T *sc = reinterpret_cast<T *>(fd2_smem);             // [CH][PW]
    T *smu = sc + CP;                                    // [EH][PW]
    T *se = smu + EP;                                    // [NE][EH][PW]
    const int tid = threadIdx.x;
    const int tx = tid & 31, ty = tid >> 5;              // warp ty owns tile rows ty and ty + 8
    const int x0 = blockIdx.x * TX, y0 = blockIdx.y * TY;
    const long rep = (long)blockIdx.z * p.N;             // replica of a batched context
    const int mx = p.nx - 1, my = p.ny - 1;
    const T rx = p.rdx2[0], ry = p.rdx2[1];

    grid_dependency_wait();
    grid_dependents_launch();

    for (int t = tid; t < CP / 2; t += 256) {
        const int row = t / (PW / 2), cp = t - row * (PW / 2);
        cp_async_pair2(sc + row * PW + 2 * cp, p.c + rep + (long)((y0 + row - 2) & my) * p.nx + ((x0 + 2 * cp - 2) & mx));
    }
#pragma unroll
    for (int f = 0; f < NE; ++f) {
        const T *src = p.eta + (long)f * p.fs + rep;
        T *dst = se + f * EP;
        for (int t = tid; t < EP / 2; t += 256) {
            const int row = t / (PW / 2), cp = t - row * (PW / 2);
            cp_async_pair2(dst + row * PW + 2 * cp, src + (long)((y0 + row - 1) & my) * p.nx + ((x0 + 2 * cp - 2) & mx));
        }
    }
    asm volatile("cp.async.wait_all;" ::: "memory");
    __syncthreads();

    auto ld2 = [](const T *q) { return *reinterpret_cast<const P2 *>(q); };
    auto lap = [&](const T *P, int o, P2 v) {            // 5-point Laplacian of the pair at offset o of plane P (pitch PW)
        const T l = P[o - 1], r = P[o + 2];
        const P2 u = ld2(P + o - PW), d = ld2(P + o + PW);
        P2 out;
        out.x = rx * (l + v.y - T(2) * v.x) + ry * (u.x + d.x - T(2) * v.x);
        out.y = rx * (v.x + r - T(2) * v.y) + ry * (u.y + d.y - T(2) * v.y);
        return out;
    };
    // kernel (i) for the pair at mu row rr (y0 - 1 + rr), column pair starting at ix
    auto mu_pair = [&](int rr, int ix, P2 v, const P2 *e) {
        const P2 l = lap(sc, (rr + 1) * PW + ix, v);
        T h0 = 0, h1 = 0;
#pragma unroll
        for (int f = 0; f < NE; ++f) { h0 += h_term(e[f].x); h1 += h_term(e[f].y); }
        P2 mu;
        mu.x = dfdc(p.m, v.x, h0) - p.m.kappa_c * l.x;
        mu.y = dfdc(p.m, v.y, h1) - p.m.kappa_c * l.y;
        *reinterpret_cast<P2 *>(smu + rr * PW + ix) = mu;
        return mu;
    };

    constexpr int NR = NE > 0 ? NE : 1;
    const int ix = 2 + 2 * tx;
    P2 cown[2], mown[2], eown[2][NR];
#pragma unroll
    for (int h = 0; h < 2; ++h) {                        // own points: tile rows ty + 8 h  ->  mu row rr = row + 1
        const int rr = ty + 8 * h + 1;
        cown[h] = ld2(sc + (rr + 1) * PW + ix);
#pragma unroll
        for (int f = 0; f < NE; ++f) eown[h][f] = ld2(se + f * EP + rr * PW + ix);
        mown[h] = mu_pair(rr, ix, cown[h], eown[h]);
    }
    if (ty < 2) {                                        // ring rows y0 - 1 and y0 + TY
        const int rr = ty ? TY + 1 : 0;
        P2 e[NR];
#pragma unroll
        for (int f = 0; f < NE; ++f) e[f] = ld2(se + f * EP + rr * PW + ix);
        mu_pair(rr, ix, ld2(sc + (rr + 1) * PW + ix), e);
    } else if (ty < 4 && tx < EH) {                      // ring columns x0 - 1 (warp 2) and x0 + TX (warp 3), single points
        const int rr = tx, col = (ty == 2) ? 1 : TX + 2;
        const int oc = (rr + 1) * PW + col, oe = rr * PW + col;
        const T v = sc[oc];
        const T l = rx * (sc[oc - 1] + sc[oc + 1] - T(2) * v) + ry * (sc[oc - PW] + sc[oc + PW] - T(2) * v);
        T h = 0;
#pragma unroll
        for (int f = 0; f < NE; ++f) h += h_term(se[f * EP + oe]);
        smu[oe] = dfdc(p.m, v, h) - p.m.kappa_c * l;
    }
    __syncthreads();

    // kernels (ii) + (iii) on the thread's own points
#pragma unroll
    for (int h = 0; h < 2; ++h) {
        const int rr = ty + 8 * h + 1, o = rr * PW + ix;
        const long g = rep + (long)(y0 + ty + 8 * h) * p.nx + (x0 + 2 * tx);
        const P2 lm = lap(smu, o, mown[h]);
        P2 cn; cn.x = cown[h].x + p.m.dtM * lm.x; cn.y = cown[h].y + p.m.dtM * lm.y;
        *reinterpret_cast<P2 *>(p.c_new + g) = cn;
        T s0 = 0, s1 = 0;
#pragma unroll
        for (int f = 0; f < NE; ++f) { s0 += eown[h][f].x * eown[h][f].x; s1 += eown[h][f].y * eown[h][f].y; }
#pragma unroll
        for (int f = 0; f < NE; ++f) {
            const P2 e = eown[h][f];
            const P2 le = lap(se + f * EP, o, e);
            P2 en;
            en.x = e.x - p.m.dtL * (dfdeta(p.m, cown[h].x, e.x, s0) - p.m.kappa_eta * le.x);
            en.y = e.y - p.m.dtL * (dfdeta(p.m, cown[h].y, e.y, s1) - p.m.kappa_eta * le.y);
            *reinterpret_cast<P2 *>(p.eta_new + (long)f * p.fs + g) = en;
        }
    }
}

template <typename T, int NE> static cudaError_t launch_fd2d_pair_ne(const FdParams<T> &p, cudaStream_t s)
{
    constexpr int PW = 68, CP = 20 * PW, EP = 18 * PW;
    const size_t smem = sizeof(T) * ((size_t)CP + (size_t)(1 + NE) * EP);
    auto kern = fd2d_pair_kernel<T, NE>;
    if (smem > 48 * 1024) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
    }
    return launch_pdl(kern, dim3((unsigned)(p.nx / 64), (unsigned)(p.ny / 16), (unsigned)(p.nbatch > 0 ? p.nbatch : 1)), dim3(256), smem, s, true, p);
}

// nx >= 64, ny >= 16, nz == 1; cudaErrorNotSupported otherwise (fd_fused2d_kernel serves those)
template <typename T> cudaError_t launch_fd2d_pair(const FdParams<T> &p, cudaStream_t s)
{
    if (p.nx < 64 || p.ny < 16 || p.nz != 1) return cudaErrorNotSupported;
    switch (p.m.n_eta) {
    case 0: return launch_fd2d_pair_ne<T, 0>(p, s);
    case 1: return launch_fd2d_pair_ne<T, 1>(p, s);
    case 2: return launch_fd2d_pair_ne<T, 2>(p, s);
    case 3: return launch_fd2d_pair_ne<T, 3>(p, s);
    case 4: return launch_fd2d_pair_ne<T, 4>(p, s);
    case 5: return launch_fd2d_pair_ne<T, 5>(p, s);
    case 6: return launch_fd2d_pair_ne<T, 6>(p, s);
    case 7: return launch_fd2d_pair_ne<T, 7>(p, s);
    case 8: return launch_fd2d_pair_ne<T, 8>(p, s);
    }
    return cudaErrorNotSupported;
}

template cudaError_t launch_fd2d_pair<double>(const FdParams<double> &, cudaStream_t);
template cudaError_t launch_fd2d_pair<float>(const FdParams<float> &, cudaStream_t);

}  // namespace pf
