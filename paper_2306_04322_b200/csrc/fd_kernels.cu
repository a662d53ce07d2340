// fd_kernels.cu -- the explicit forward-Euler finite-difference step
// and the real-space part of the free-energy functional (Eq. 1).
//
// Paper form: kernel (i) mu = df/dc - kappa_c lap c, kernel (ii) c' = c + dt M lap mu, kernel (iii)
// eta_i' = eta_i - dt L (df/deta_i - kappa_eta lap eta_i); 2nd-order centred 5-point (2D) / 7-point (3D)
// Laplacian, periodic boundaries, every right-hand side at time t. The ghost layers are replaced by wrap-around
// index arithmetic (no ghost storage).
//   2D: ONE launch per step. A CTA stages a TX x TY tile in shared memory -- c with a halo of two points, every
//       eta_i with a halo of one -- forms mu on the tile plus a ring of one point (kernel (i)), and from that
//       the new c and eta_i of the tile (kernels (ii), (iii)): each field is read once and written once per step,
//       2(p+1) R bytes instead of the (3p+5) R of the separate kernels (the halo re-reads stay in L1/L2).
//   3D: kernels (i) and (ii)+(iii) as two launches on global memory (neighbours served by L1/L2).
#include "pf_kernels.cuh"

#ifndef PF_FD_TY
#define PF_FD_TY 16
#endif

namespace pf {

struct Nbr { long xm, xp, ym, yp, zm, zp; };

// global -> shared copy of one element without a register stop-over (LDGSTS): a thread queues all of its tile
// elements at once and waits once, so a CTA has its whole tile in flight
template <typename T> __device__ __forceinline__ void cp_async_elem(T *smem_dst, const T *gmem_src)
{
    asm volatile("cp.async.ca.shared.global [%0], [%1], %2;" ::"r"((unsigned)__cvta_generic_to_shared(smem_dst)), "l"(gmem_src), "n"(sizeof(T)) : "memory");
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }

__device__ __forceinline__ Nbr neighbours(long i, int nx, int ny, int nz)
{
    const int x = (int)(i % nx);
    const long r = i / nx;
    const int y = (int)(r % ny);
    const int z = (int)(r / ny);
    Nbr n;
    n.xm = i + (x == 0 ? nx - 1 : -1);
    n.xp = i + (x == nx - 1 ? -(nx - 1) : 1);
    n.ym = i + (y == 0 ? (long)(ny - 1) * nx : -(long)nx);
    n.yp = i + (y == ny - 1 ? -(long)(ny - 1) * nx : (long)nx);
    const long pl = (long)nx * ny;
    n.zm = i + (z == 0 ? (long)(nz - 1) * pl : -pl);
    n.zp = i + (z == nz - 1 ? -(long)(nz - 1) * pl : pl);
    return n;
}

template <typename T>
__device__ __forceinline__ T lap(const T *__restrict__ u, long i, const Nbr &n, const T (&rdx2)[3], bool threeD)
{
    const T v = u[i];
    T s = rdx2[0] * (u[n.xp] + u[n.xm] - T(2) * v) + rdx2[1] * (u[n.yp] + u[n.ym] - T(2) * v);
    if (threeD) s += rdx2[2] * (u[n.zp] + u[n.zm] - T(2) * v);
    return s;
}

// kernel (i): mu = df_chem/dc - kappa_c lap c
template <typename T> __global__ void fd_mu_kernel(const FdParams<T> p)
{
    const long i = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= p.N) return;
    const Nbr n = neighbours(i, p.nx, p.ny, p.nz);
    T h = 0;
    for (int k = 0; k < p.m.n_eta; ++k) h += h_term(p.eta[(long)k * p.N + i]);
    p.mu[i] = dfdc(p.m, p.c[i], h) - p.m.kappa_c * lap(p.c, i, n, p.rdx2, p.nz > 1);
}

// kernels (ii) + (iii)
template <typename T> __global__ void fd_update_kernel(const FdParams<T> p)
{
    const long i = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= p.N) return;
    const bool threeD = p.nz > 1;
    const Nbr n = neighbours(i, p.nx, p.ny, p.nz);
    const T c = p.c[i];
    p.c_new[i] = c + p.m.dtM * lap(p.mu, i, n, p.rdx2, threeD);
    T s2 = 0;
    for (int k = 0; k < p.m.n_eta; ++k) { const T e = p.eta[(long)k * p.N + i]; s2 += e * e; }
    for (int k = 0; k < p.m.n_eta; ++k) {
        const T *e = p.eta + (long)k * p.N;
        p.eta_new[(long)k * p.N + i] = e[i] - p.m.dtL * (dfdeta(p.m, c, e[i], s2) - p.m.kappa_eta * lap(e, i, n, p.rdx2, threeD));
    }
}

// 2D fused step, see the header. Dynamic shared memory: c tile (TY+4) x (TX+4), mu tile (TY+2) x (TX+2),
// n_eta tiles (TY+2) x (TX+2). nx, ny are powers of two >= TX, TY.
template <typename T, int TX, int TY, int NE>
__global__ void __launch_bounds__(256) fd_fused2d_kernel(const FdParams<T> p)
{
    constexpr int CW = TX + 4, CH = TY + 4, EW = TX + 2, EH = TY + 2;
    extern __shared__ __align__(16) unsigned char fd_smem[];
    T *sc = reinterpret_cast<T *>(fd_smem);
    T *smu = sc + CW * CH;
    T *se = smu + EW * EH;
    const int x0 = blockIdx.x * TX, y0 = blockIdx.y * TY;
    const int mx = p.nx - 1, my = p.ny - 1;
    constexpr int ne = NE;                 // compile-time field count: the per-field loops unroll into fixed offsets

    // thread (tx, ty) of TX x (256/TX): column tx (+ the halo columns for the first lanes), rows ty, ty + TYS, ..
    constexpr int TYS = 256 / TX;
    const int tx = threadIdx.x % TX, ty = threadIdx.x / TX;
    grid_dependency_wait();
    grid_dependents_launch();

    for (int ly = ty; ly < CH; ly += TYS) {
        const T *row = p.c + (long)((y0 + ly - 2) & my) * p.nx;
        cp_async_elem(sc + ly * CW + tx, row + ((x0 + tx - 2) & mx));
        if (tx < 4) cp_async_elem(sc + ly * CW + TX + tx, row + ((x0 + TX + tx - 2) & mx));
    }
    for (int k = 0; k < ne; ++k) {
        const T *ek = p.eta + (long)k * p.N;
        T *sk = se + k * (EW * EH);
        for (int ly = ty; ly < EH; ly += TYS) {
            const T *row = ek + (long)((y0 + ly - 1) & my) * p.nx;
            cp_async_elem(sk + ly * EW + tx, row + ((x0 + tx - 1) & mx));
            if (tx < 2) cp_async_elem(sk + ly * EW + TX + tx, row + ((x0 + TX + tx - 1) & mx));
        }
    }
    cp_async_wait_all();
    __syncthreads();

    // kernel (i) on the tile and its ring: mu = df_chem/dc - kappa_c lap c
    auto mu_at = [&](int lx, int ly) {
        const int i = ly * EW + lx;
        const T *cc = sc + (ly + 1) * CW + (lx + 1);
        const T v = cc[0];
        const T l = p.rdx2[0] * (cc[1] + cc[-1] - T(2) * v) + p.rdx2[1] * (cc[CW] + cc[-CW] - T(2) * v);
        T h = 0;
        for (int k = 0; k < ne; ++k) h += h_term(se[k * (EW * EH) + i]);
        smu[i] = dfdc(p.m, v, h) - p.m.kappa_c * l;
    };
    for (int ly = ty; ly < EH; ly += TYS) {
        mu_at(tx, ly);
        if (tx < 2) mu_at(TX + tx, ly);
    }
    __syncthreads();

    // kernels (ii) + (iii) on the tile
    for (int ly = ty; ly < TY; ly += TYS) {
        const int lx = tx;
        const long g = (long)(y0 + ly) * p.nx + (x0 + lx);
        const int e0 = (ly + 1) * EW + (lx + 1);
        const T c = sc[(ly + 2) * CW + (lx + 2)];
        const T *mu = smu + e0;
        const T lm = p.rdx2[0] * (mu[1] + mu[-1] - T(2) * mu[0]) + p.rdx2[1] * (mu[EW] + mu[-EW] - T(2) * mu[0]);
        p.c_new[g] = c + p.m.dtM * lm;
        T s2 = 0;
        for (int k = 0; k < ne; ++k) { const T e = se[k * (EW * EH) + e0]; s2 += e * e; }
        for (int k = 0; k < ne; ++k) {
            const T *e = se + k * (EW * EH) + e0;
            const T le = p.rdx2[0] * (e[1] + e[-1] - T(2) * e[0]) + p.rdx2[1] * (e[EW] + e[-EW] - T(2) * e[0]);
            p.eta_new[(long)k * p.N + g] = e[0] - p.m.dtL * (dfdeta(p.m, c, e[0], s2) - p.m.kappa_eta * le);
        }
    }
}

// Eq. 1 pieces in real space: acc[0] += sum f_chem, acc[1] += sum |grad c|^2, acc[2+i] += sum |grad eta_i|^2
// (forward differences when gradient_kind == 1). Accumulated in fp64; scaled by the caller.
template <typename T> __global__ void energy_kernel(const EnergyParams<T> p)
{
    __shared__ double red[32];
    const int nacc = 2 + p.m.n_eta;
    double part[2 + 8];
    for (int a = 0; a < nacc; ++a) part[a] = 0.0;
    for (long i = (long)blockIdx.x * blockDim.x + threadIdx.x; i < p.N; i += (long)gridDim.x * blockDim.x) {
        const Nbr n = neighbours(i, p.nx, p.ny, p.nz);
        const T c = p.c[i];
        T h = 0, g = 0, s2 = 0, s4 = 0;
        for (int k = 0; k < p.m.n_eta; ++k) {
            const T e = p.eta[(long)k * p.N + i];
            h += h_term(e);
            g += e * e * (T(1) - e) * (T(1) - e);
            s2 += e * e; s4 += e * e * e * e;
        }
        g += p.m.alpha * (s2 * s2 - s4);               // sum_i sum_{j != i} eta_i^2 eta_j^2
        const T fa = p.m.rho2 * (c - p.m.c_alpha) * (c - p.m.c_alpha);
        const T fb = p.m.rho2 * (p.m.c_beta - c) * (p.m.c_beta - c);
        part[0] += (double)(fa * (T(1) - h) + fb * h + p.m.w * g);
        if (p.gradient_kind == 1) {
            for (int k = -1; k < p.m.n_eta; ++k) {
                const T *u = (k < 0) ? p.c : p.eta + (long)k * p.N;
                const T u0 = u[i];
                const T gx = (u[n.xp] - u0) * p.rdx[0], gy = (u[n.yp] - u0) * p.rdx[1];
                const T gz = (p.nz > 1) ? (u[n.zp] - u0) * p.rdx[2] : T(0);
                part[2 + k] += (double)gx * gx + (double)gy * gy + (double)gz * gz;
            }
        }
    }
    for (int a = 0; a < nacc; ++a) {
        double v = part[a];
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        __syncthreads();
        if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = v;
        __syncthreads();
        if (threadIdx.x == 0) {
            double tot = 0.0;
            for (int w = 0; w < (int)(blockDim.x >> 5); ++w) tot += red[w];
            atomicAdd(p.acc + a, tot);
        }
    }
}

template <typename T> cudaError_t launch_fd_mu(const FdParams<T> &p, cudaStream_t s)
{
    fd_mu_kernel<T><<<(unsigned)((p.N + 255) / 256), 256, 0, s>>>(p);
    return cudaGetLastError();
}
template <typename T> cudaError_t launch_fd_update(const FdParams<T> &p, cudaStream_t s)
{
    fd_update_kernel<T><<<(unsigned)((p.N + 255) / 256), 256, 0, s>>>(p);
    return cudaGetLastError();
}
template <typename T, int TX, int TY, int NE> static cudaError_t launch_fd_fused2d_ne(const FdParams<T> &p, cudaStream_t s)
{
    const size_t smem = sizeof(T) * ((size_t)(TX + 4) * (TY + 4) + (size_t)(1 + NE) * (TX + 2) * (TY + 2));
    auto kern = fd_fused2d_kernel<T, TX, TY, NE>;
    if (smem > 48 * 1024) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
    }
    // programmatic dependent launch: consecutive steps cannot overlap, but the launch latency of step t+1 hides
    // behind the tail of step t
    return launch_pdl(kern, dim3((unsigned)(p.nx / TX), (unsigned)(p.ny / TY)), dim3(256), smem, s, true, p);
}
template <typename T, int TX, int TY> static cudaError_t launch_fd_fused2d_inst(const FdParams<T> &p, cudaStream_t s)
{
    switch (p.m.n_eta) {
    case 0: return launch_fd_fused2d_ne<T, TX, TY, 0>(p, s);
    case 1: return launch_fd_fused2d_ne<T, TX, TY, 1>(p, s);
    case 2: return launch_fd_fused2d_ne<T, TX, TY, 2>(p, s);
    case 3: return launch_fd_fused2d_ne<T, TX, TY, 3>(p, s);
    case 4: return launch_fd_fused2d_ne<T, TX, TY, 4>(p, s);
    case 5: return launch_fd_fused2d_ne<T, TX, TY, 5>(p, s);
    case 6: return launch_fd_fused2d_ne<T, TX, TY, 6>(p, s);
    case 7: return launch_fd_fused2d_ne<T, TX, TY, 7>(p, s);
    case 8: return launch_fd_fused2d_ne<T, TX, TY, 8>(p, s);
    }
    return cudaErrorInvalidValue;
}
// one fused launch per 2D step (nz == 1)
template <typename T> cudaError_t launch_fd_fused2d(const FdParams<T> &p, cudaStream_t s)
{
    if (p.nx >= 64) return launch_fd_fused2d_inst<T, 64, PF_FD_TY>(p, s);
    if (p.nx >= 32) return launch_fd_fused2d_inst<T, 32, PF_FD_TY>(p, s);
    return launch_fd_fused2d_inst<T, 16, 16>(p, s);
}
template <typename T> cudaError_t launch_energy(const EnergyParams<T> &p, cudaStream_t s)
{
    long blocks = (p.N + 255) / 256;
    if (blocks > 148 * 8) blocks = 148 * 8;
    energy_kernel<T><<<(unsigned)blocks, 256, 0, s>>>(p);
    return cudaGetLastError();
}

template cudaError_t launch_fd_mu<double>(const FdParams<double> &, cudaStream_t);
template cudaError_t launch_fd_mu<float>(const FdParams<float> &, cudaStream_t);
template cudaError_t launch_fd_update<double>(const FdParams<double> &, cudaStream_t);
template cudaError_t launch_fd_update<float>(const FdParams<float> &, cudaStream_t);
template cudaError_t launch_fd_fused2d<double>(const FdParams<double> &, cudaStream_t);
template cudaError_t launch_fd_fused2d<float>(const FdParams<float> &, cudaStream_t);
template cudaError_t launch_energy<double>(const EnergyParams<double> &, cudaStream_t);
template cudaError_t launch_energy<float>(const EnergyParams<float> &, cudaStream_t);

}  // namespace pf
