// fd_kernels.cu -- the explicit forward-Euler finite-difference step
// and the real-space part of the free-energy functional (Eq. 1).
//
// Paper form: kernel (i) mu = df/dc - kappa_c lap c, kernel (ii) c' = c + dt M lap mu, kernel (iii)
// eta_i' = eta_i - dt L (df/deta_i - kappa_eta lap eta_i); 2nd-order centred 5-point (2D) / 7-point (3D)
// Laplacian, periodic boundaries, every right-hand side at time t. Here (ii) and (iii) are one launch
// and the ghost layers are replaced by wrap-around index arithmetic (no ghost storage).
#include "pf_kernels.cuh"

namespace pf {

struct Nbr { long xm, xp, ym, yp, zm, zp; };

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
template cudaError_t launch_energy<double>(const EnergyParams<double> &, cudaStream_t);
template cudaError_t launch_energy<float>(const EnergyParams<float> &, cudaStream_t);

}  // namespace pf
