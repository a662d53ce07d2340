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
//   3D: ONE launch per step as well: a CTA marches along z with rings of planes in shared memory (fd_fused3d_kernel).
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
    const long rep = (long)blockIdx.z * p.N;             // replica of a batched context
    const int mx = p.nx - 1, my = p.ny - 1;
    constexpr int ne = NE;                 // compile-time field count: the per-field loops unroll into fixed offsets

    // thread (tx, ty) of TX x (256/TX): column tx (+ the halo columns for the first lanes), rows ty, ty + TYS, ..
    constexpr int TYS = 256 / TX;
    const int tx = threadIdx.x % TX, ty = threadIdx.x / TX;
    grid_dependency_wait();
    grid_dependents_launch();

    for (int ly = ty; ly < CH; ly += TYS) {
        const T *row = p.c + rep + (long)((y0 + ly - 2) & my) * p.nx;
        cp_async_elem(sc + ly * CW + tx, row + ((x0 + tx - 2) & mx));
        if (tx < 4) cp_async_elem(sc + ly * CW + TX + tx, row + ((x0 + TX + tx - 2) & mx));
    }
    for (int k = 0; k < ne; ++k) {
        const T *ek = p.eta + (long)k * p.fs + rep;
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
        const long g = rep + (long)(y0 + ly) * p.nx + (x0 + lx);
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
            p.eta_new[(long)k * p.fs + g] = e[0] - p.m.dtL * (dfdeta(p.m, c, e[0], s2) - p.m.kappa_eta * le);
        }
    }
}

// 3D fused step: a CTA owns a TX x TY tile of (x, y) and marches along z over a chunk of zc planes, keeping in shared
// memory rings of the last planes it needs: c (halo 2 in x, y; 4 slots), every eta_i (halo 1; 4 slots) and mu (tile +
// ring of one point; 3 slots). Per output plane k: queue c(k+2), eta(k+1) with cp.async; form mu(k+1) from c(k..k+2) and
// eta(k+1); then c', eta' of plane k from mu(k-1..k+1), eta(k-1..k+1). Each field is read about once ((1 + halo) x
// (1 + 4/zc)) and written once per step instead of the (3p+5) R of the two global-memory kernels. Two barriers per plane:
// the 4-slot rings make the next plane's loads land in slots no thread still reads.
template <typename T, int TX, int TY, int NE>
__global__ void __launch_bounds__(TX * TY) fd_fused3d_kernel(const FdParams<T> p, const int zc)
{
    constexpr int CW = TX + 4, CH = TY + 4, EW = TX + 2, EH = TY + 2, CP = CW * CH, EP = EW * EH;
    extern __shared__ __align__(16) unsigned char fd_smem[];
    T *sc = reinterpret_cast<T *>(fd_smem);          // [4][CP]
    T *smu = sc + 4 * CP;                            // [3][EP]
    T *se = smu + 3 * EP;                            // [NE][4][EP]
    const int x0 = blockIdx.x * TX, y0 = blockIdx.y * TY, z0 = blockIdx.z * zc;
    const int mx = p.nx - 1, my = p.ny - 1, mz = p.nz - 1;
    const long plane = (long)p.nx * p.ny;
    const int tx = threadIdx.x % TX, ty = threadIdx.x / TX;

    auto load_c = [&](int m) {                       // plane z0 + m -> slot m & 3
        const T *src = p.c + (long)((z0 + m) & mz) * plane;
        T *dst = sc + ((m + 4) & 3) * CP;
        for (int ly = ty; ly < CH; ly += TY) {
            const T *row = src + (long)((y0 + ly - 2) & my) * p.nx;
            cp_async_elem(dst + ly * CW + tx, row + ((x0 + tx - 2) & mx));
            if (tx < 4) cp_async_elem(dst + ly * CW + TX + tx, row + ((x0 + TX + tx - 2) & mx));
        }
    };
    auto load_e = [&](int m) {
        for (int k = 0; k < NE; ++k) {
            const T *src = p.eta + (long)k * p.fs + (long)((z0 + m) & mz) * plane;
            T *dst = se + (k * 4 + ((m + 4) & 3)) * EP;
            for (int ly = ty; ly < EH; ly += TY) {
                const T *row = src + (long)((y0 + ly - 1) & my) * p.nx;
                cp_async_elem(dst + ly * EW + tx, row + ((x0 + tx - 1) & mx));
                if (tx < 2) cp_async_elem(dst + ly * EW + TX + tx, row + ((x0 + TX + tx - 1) & mx));
            }
        }
    };
    // kernel (i) for plane m on the tile and its ring; slot3 = m mod 3 kept by the caller
    auto mu_plane = [&](int m, int slot3) {
        const T *c0 = sc + ((m + 4) & 3) * CP, *cm = sc + ((m + 3) & 3) * CP, *cp = sc + ((m + 5) & 3) * CP;
        T *mu = smu + slot3 * EP;
        auto at = [&](int lx, int ly) {
            const int i = ly * EW + lx, ci = (ly + 1) * CW + (lx + 1);
            const T v = c0[ci];
            const T l = p.rdx2[0] * (c0[ci + 1] + c0[ci - 1] - T(2) * v) + p.rdx2[1] * (c0[ci + CW] + c0[ci - CW] - T(2) * v)
                      + p.rdx2[2] * (cp[ci] + cm[ci] - T(2) * v);
            T h = 0;
            for (int k = 0; k < NE; ++k) h += h_term(se[(k * 4 + ((m + 4) & 3)) * EP + i]);
            mu[i] = dfdc(p.m, v, h) - p.m.kappa_c * l;
        };
        for (int ly = ty; ly < EH; ly += TY) {
            at(tx, ly);
            if (tx < 2) at(TX + tx, ly);
        }
    };

    grid_dependency_wait();
    grid_dependents_launch();

    // prologue: mu(-1) and mu(0)
    load_c(-2); load_c(-1); load_c(0); load_e(-1); load_e(0);
    cp_async_wait_all();
    __syncthreads();
    mu_plane(-1, 2);
    load_c(1);                                       // slot of c(-3): free
    cp_async_wait_all();
    __syncthreads();
    mu_plane(0, 0);
    // no barrier needed here: the loop starts with loads into free slots and a barrier before mu(k+1) is formed

    int s3 = 0;                                      // k mod 3
    for (int k = 0; k < zc; ++k) {
        load_c(k + 2);                               // slot of c(k-2)
        load_e(k + 1);                               // slot of eta(k-3)
        cp_async_wait_all();
        __syncthreads();
        const int s3p = (s3 == 2) ? 0 : s3 + 1, s3m = (s3 == 0) ? 2 : s3 - 1;
        mu_plane(k + 1, s3p);                        // overwrites mu(k-2)
        __syncthreads();

        // kernels (ii) + (iii) on plane k
        const int e0 = (ty + 1) * EW + (tx + 1);
        const long g = (long)((z0 + k) & mz) * plane + (long)(y0 + ty) * p.nx + (x0 + tx);
        const T c = sc[((k + 4) & 3) * CP + (ty + 2) * CW + (tx + 2)];
        const T *mu = smu + s3 * EP + e0;
        const T lm = p.rdx2[0] * (mu[1] + mu[-1] - T(2) * mu[0]) + p.rdx2[1] * (mu[EW] + mu[-EW] - T(2) * mu[0])
                   + p.rdx2[2] * (smu[s3p * EP + e0] + smu[s3m * EP + e0] - T(2) * mu[0]);
        p.c_new[g] = c + p.m.dtM * lm;
        T s2 = 0;
        for (int f = 0; f < NE; ++f) { const T e = se[(f * 4 + ((k + 4) & 3)) * EP + e0]; s2 += e * e; }
        for (int f = 0; f < NE; ++f) {
            const T *e = se + (f * 4 + ((k + 4) & 3)) * EP + e0;
            const T ezp = se[(f * 4 + ((k + 5) & 3)) * EP + e0], ezm = se[(f * 4 + ((k + 3) & 3)) * EP + e0];
            const T le = p.rdx2[0] * (e[1] + e[-1] - T(2) * e[0]) + p.rdx2[1] * (e[EW] + e[-EW] - T(2) * e[0])
                       + p.rdx2[2] * (ezp + ezm - T(2) * e[0]);
            p.eta_new[(long)f * p.fs + g] = e[0] - p.m.dtL * (dfdeta(p.m, c, e[0], s2) - p.m.kappa_eta * le);
        }
        s3 = s3p;
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
    return launch_pdl(kern, dim3((unsigned)(p.nx / TX), (unsigned)(p.ny / TY), (unsigned)(p.nbatch > 0 ? p.nbatch : 1)), dim3(256), smem, s, true, p);
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
template <typename T, int TX, int TY, int NE> static cudaError_t launch_fd_fused3d_ne(const FdParams<T> &p, cudaStream_t s)
{
    const size_t smem = sizeof(T) * ((size_t)4 * (TX + 4) * (TY + 4) + (size_t)(3 + 4 * NE) * (TX + 2) * (TY + 2));
    auto kern = fd_fused3d_kernel<T, TX, TY, NE>;
    if (smem > 48 * 1024) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
    }
    // chunks along z: enough CTAs for ~8 per SM, at least 16 planes per chunk (4 extra planes are read per chunk)
    const int tiles = (p.nx / TX) * (p.ny / TY);
    int chunks = 1;
    while (tiles * chunks < 1184 && p.nz / (2 * chunks) >= 16) chunks *= 2;
    const int zc = p.nz / chunks;
    return launch_pdl(kern, dim3((unsigned)(p.nx / TX), (unsigned)(p.ny / TY), (unsigned)chunks), dim3(TX * TY), smem, s, true, p, zc);
}
template <typename T, int TX, int TY> static cudaError_t launch_fd_fused3d_inst(const FdParams<T> &p, cudaStream_t s)
{
    switch (p.m.n_eta) {
    case 0: return launch_fd_fused3d_ne<T, TX, TY, 0>(p, s);
    case 1: return launch_fd_fused3d_ne<T, TX, TY, 1>(p, s);
    case 2: return launch_fd_fused3d_ne<T, TX, TY, 2>(p, s);
    case 3: return launch_fd_fused3d_ne<T, TX, TY, 3>(p, s);
    case 4: return launch_fd_fused3d_ne<T, TX, TY, 4>(p, s);
    case 5: return launch_fd_fused3d_ne<T, TX, TY, 5>(p, s);
    case 6: return launch_fd_fused3d_ne<T, TX, TY, 6>(p, s);
    case 7: return launch_fd_fused3d_ne<T, TX, TY, 7>(p, s);
    case 8: return launch_fd_fused3d_ne<T, TX, TY, 8>(p, s);
    }
    return cudaErrorInvalidValue;
}
// one fused launch per 3D step
template <typename T> cudaError_t launch_fd_fused3d(const FdParams<T> &p, cudaStream_t s)
{
    if (p.nx >= 32) return launch_fd_fused3d_inst<T, 32, 8>(p, s);
    return launch_fd_fused3d_inst<T, 16, 16>(p, s);
}
template <typename T> cudaError_t launch_energy(const EnergyParams<T> &p, cudaStream_t s)
{
    long blocks = (p.N + 255) / 256;
    if (blocks > 148 * 8) blocks = 148 * 8;
    energy_kernel<T><<<(unsigned)blocks, 256, 0, s>>>(p);
    return cudaGetLastError();
}

template cudaError_t launch_fd_fused3d<double>(const FdParams<double> &, cudaStream_t);
template cudaError_t launch_fd_fused3d<float>(const FdParams<float> &, cudaStream_t);
template cudaError_t launch_fd_fused2d<double>(const FdParams<double> &, cudaStream_t);
template cudaError_t launch_fd_fused2d<float>(const FdParams<float> &, cudaStream_t);
template cudaError_t launch_energy<double>(const EnergyParams<double> &, cudaStream_t);
template cudaError_t launch_energy<float>(const EnergyParams<float> &, cudaStream_t);

}  // namespace pf
