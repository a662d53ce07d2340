// static_energy.cu -- pf_free_energy_static (include/pf.h): the real-space free energy of Eq. 1 for
// callers that must not allocate device memory.
//
// Who this is for. pf_create reserves every buffer a context needs with cudaMalloc, and pf_free_energy lives on such a
// context. Some programs cannot afford that call at the point where they want the energy:
//   * a host application that has handed (nearly) all device memory to a pool of its own -- a framework's caching
//     allocator, a solver with a fixed memory budget -- so a cudaMalloc from a plug-in fails or eats into a budget the
//     plug-in does not own;
//   * an in-situ monitor called from inside somebody else's time loop, where cudaMalloc / cudaFree would stall the whole
//     device (both synchronise it) every time the monitor runs;
//   * code under a "no allocation after start-up" rule (long-running services that must not fragment or fail late).
// This entry point takes the fields where they already are (device pointers of the caller), needs no context, and gets
// the little working memory it needs -- per-tile partial sums, a ticket and the result -- from ONE array that is part
// of the library image itself: g_energy_scratch below, PF_STATIC_SCRATCH_BYTES (about 320 KB) of global memory that
// every GPU holds from the moment it loads libpf.so until the process ends, whether the entry point is used or not.
// That array is the reason for the size limit: PF_STATIC_MAX_POINTS grid points, 8 order parameters.
//
// The kernel is a variant of energy_kernel (fd_kernels.cu): same pointwise arithmetic, same fp64 accumulation, but
// instead of atomics on a context's accumulator each CTA sums a fixed tile of PF_STATIC_TILE points and parks its
// partial sums in the static array; the CTA that finishes last adds them up in tile order. The result therefore does
// not depend on the number of SMs or on the order in which CTAs retire (bit-reproducible).
//
// Rules that follow from "one shared array":
//   * the array keeps whatever the previous call left in it. The ticket and the result slots must start at zero and
//     are cleared on the caller's stream at the head of every call; the partial sums are overwritten before they are read;
//   * two calls whose GPU work overlaps -- different streams, different host threads -- race on the array and give
//     garbage. Calls on one stream are safe (they are ordered). Host-side, the set-up below is guarded by a mutex; the
//     GPU work is not, on purpose;
//   * the name g_energy_scratch means something else in host code than in device code: on the host it is only a
//     handle for the runtime, not an address the GPU could use. The address is fetched once per device with
//     cudaGetSymbolAddress, with that device current, by the first call made on that device. That first call
//     should therefore be made during start-up, before any stream capture begins.
// No cudaMalloc, cudaFree, stream/event creation or other allocating runtime call is made here.
#include <mutex>

#include "../../include/pf.h"
#include "pf_kernels.cuh"

namespace {

constexpr int kTile = PF_STATIC_TILE;                       // grid points per CTA
constexpr int kThreads = 256;
constexpr int kPerThread = kTile / kThreads;
constexpr int kMaxTiles = PF_STATIC_MAX_POINTS / PF_STATIC_TILE;
constexpr int kMaxAcc = 2 + 8;                              // chemical, |grad c|^2, |grad eta_i|^2 for up to 8 eta
constexpr int kHead = 32;                                   // doubles: [0] ticket (as unsigned), [16 .. 16+kMaxAcc) result
constexpr int kResult = 16;
constexpr size_t kScratchDoubles = (size_t)kHead + (size_t)kMaxTiles * kMaxAcc;
static_assert(kScratchDoubles * sizeof(double) == PF_STATIC_SCRATCH_BYTES, "pf.h states the size of the static array");
static_assert(kTile % kThreads == 0, "a tile is a whole number of points per thread");

// The working memory of pf_free_energy_static. Device code may name it directly; host code must not pass this name to
// a kernel or a memset -- see scratch_of_current_device().
static __device__ __align__(256) double g_energy_scratch[kScratchDoubles];

template <typename T> struct StaticEnergyParams {
    const T *c, *eta;            // caller's device arrays: [nz][ny][nx], [n_eta][nz][ny][nx]
    int      nx, ny, nz, n_eta;
    long     N;
    T        rdx[3];             // 1/dx per axis (0 in z for 2D)
    T        rho2, c_alpha, c_beta, w, alpha;
    double  *scratch;            // device address of g_energy_scratch on the device the kernel runs on
};

// One CTA per tile of kTile consecutive grid points. part[0] = sum f_chem, part[1] = sum |grad c|^2,
// part[2+i] = sum |grad eta_i|^2 with forward differences and periodic wrap-around; f_chem as in PAPER.md:46.
template <typename T> __global__ void __launch_bounds__(kThreads) static_energy_kernel(const StaticEnergyParams<T> p)
{
    __shared__ double red[kThreads / 32][kMaxAcc];
    __shared__ bool last;
    const int nacc = 2 + p.n_eta;
    double part[kMaxAcc];
#pragma unroll
    for (int a = 0; a < kMaxAcc; ++a) part[a] = 0.0;
    const long base = (long)blockIdx.x * kTile;
    const long plane = (long)p.nx * p.ny;
    for (int j = 0; j < kPerThread; ++j) {
        const long i = base + (long)j * kThreads + threadIdx.x;
        if (i >= p.N) break;
        const int x = (int)(i % p.nx);
        const long r = i / p.nx;
        const int y = (int)(r % p.ny), z = (int)(r / p.ny);
        const long xp = i + (x == p.nx - 1 ? -(long)(p.nx - 1) : 1);
        const long yp = i + (y == p.ny - 1 ? -(long)(p.ny - 1) * p.nx : (long)p.nx);
        const long zp = i + (z == p.nz - 1 ? -(long)(p.nz - 1) * plane : plane);
        const T c = p.c[i];
        T h = 0, g = 0, s2 = 0, s4 = 0;
        for (int k = 0; k < p.n_eta; ++k) {
            const T e = p.eta[(long)k * p.N + i];
            h += pf::h_term(e);
            g += e * e * (T(1) - e) * (T(1) - e);
            s2 += e * e; s4 += e * e * e * e;
        }
        g += p.alpha * (s2 * s2 - s4);                  // sum_i sum_{j != i} eta_i^2 eta_j^2
        const T fa = p.rho2 * (c - p.c_alpha) * (c - p.c_alpha);
        const T fb = p.rho2 * (p.c_beta - c) * (p.c_beta - c);
        part[0] += (double)(fa * (T(1) - h) + fb * h + p.w * g);
#pragma unroll
        for (int k = -1; k < 8; ++k) {
            if (k >= p.n_eta) break;
            const T *u = (k < 0) ? p.c : p.eta + (long)k * p.N;
            const T u0 = u[i];
            const T gx = (u[xp] - u0) * p.rdx[0], gy = (u[yp] - u0) * p.rdx[1];
            const T gz = (p.nz > 1) ? (u[zp] - u0) * p.rdx[2] : T(0);
            part[2 + k] += (double)gx * gx + (double)gy * gy + (double)gz * gz;
        }
    }
    // CTA sum in a fixed order: lanes by butterfly, warps one after the other
#pragma unroll
    for (int a = 0; a < kMaxAcc; ++a) {
        double v = part[a];
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5][a] = v;
    }
    __syncthreads();
    double *partial = p.scratch + kHead;
    if (threadIdx.x < nacc) {
        double tot = 0.0;
        for (int w = 0; w < kThreads / 32; ++w) tot += red[w][threadIdx.x];
        partial[(size_t)blockIdx.x * kMaxAcc + threadIdx.x] = tot;
        __threadfence();                                // the partial sums are visible before the ticket is taken
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        __threadfence();
        const unsigned t = atomicAdd(reinterpret_cast<unsigned *>(p.scratch), 1u);
        last = (t == gridDim.x - 1);
    }
    __syncthreads();
    if (!last) return;
    // the CTA that retires last: one warp per accumulator, lanes stride over the tiles in tile order
    __threadfence();
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    for (int a = warp; a < nacc; a += kThreads / 32) {
        double v = 0.0;
        for (unsigned t = lane; t < gridDim.x; t += 32) v += __ldcg(partial + (size_t)t * kMaxAcc + a);
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        if (lane == 0) p.scratch[kResult + a] = v;
    }
}

// Device address of g_energy_scratch on the CURRENT device. Looked up once per device (the array exists separately on
// every GPU that loaded the library, at a different address each), remembered afterwards.
constexpr int kMaxDevices = 64;
std::mutex g_setup_mutex;
double *g_scratch_addr[kMaxDevices] = {};

int scratch_of_current_device(double **out)
{
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); return PF_ECUDA; }
    if (dev < 0 || dev >= kMaxDevices) return PF_EUNSUPPORTED;
    std::lock_guard<std::mutex> lock(g_setup_mutex);
    if (!g_scratch_addr[dev]) {
        double *ptr = nullptr;
        if (cudaGetSymbolAddress((void **)&ptr, g_energy_scratch) != cudaSuccess || !ptr) { cudaGetLastError(); return PF_ECUDA; }
        g_scratch_addr[dev] = ptr;
    }
    *out = g_scratch_addr[dev];
    return PF_OK;
}

// is `ptr` memory the current device's kernels may read (device or managed memory)?
bool device_readable(const void *ptr, int dev)
{
    cudaPointerAttributes at;
    if (cudaPointerGetAttributes(&at, ptr) != cudaSuccess) { cudaGetLastError(); return false; }
    if (at.type == cudaMemoryTypeManaged) return true;
    return at.type == cudaMemoryTypeDevice && at.device == dev;
}

template <typename T> int run(const pf_params *p, const void *c, const void *eta, long N, double *scratch, double *out)
{
    cudaStream_t s = (cudaStream_t)p->stream;
    StaticEnergyParams<T> q;
    q.c = (const T *)c; q.eta = (const T *)eta;
    q.nx = p->n[0]; q.ny = p->n[1]; q.nz = (p->ndim == 3) ? p->n[2] : 1; q.n_eta = p->n_eta; q.N = N;
    for (int d = 0; d < 3; ++d) q.rdx[d] = (d < p->ndim) ? (T)(1.0 / p->dx[d]) : (T)0;
    q.rho2 = (T)p->rho2; q.c_alpha = (T)p->c_alpha; q.c_beta = (T)p->c_beta; q.w = (T)p->w; q.alpha = (T)p->alpha;
    q.scratch = scratch;
    const unsigned tiles = (unsigned)((N + kTile - 1) / kTile);
    // ticket and result slots start at zero; whatever an earlier call (or an aborted one) left there goes
    if (cudaMemsetAsync(scratch, 0, sizeof(double) * kHead, s) != cudaSuccess) { cudaGetLastError(); return PF_ECUDA; }
    static_energy_kernel<T><<<tiles, kThreads, 0, s>>>(q);
    if (cudaGetLastError() != cudaSuccess) return PF_ECUDA;
    double h[kMaxAcc];
    const int nacc = 2 + p->n_eta;
    if (cudaMemcpyAsync(h, scratch + kResult, sizeof(double) * nacc, cudaMemcpyDeviceToHost, s) != cudaSuccess ||
        cudaStreamSynchronize(s) != cudaSuccess) { cudaGetLastError(); return PF_ECUDA; }
    double dV = 1.0;
    for (int d = 0; d < p->ndim; ++d) dV *= p->dx[d];
    out[1] = h[0] * dV;
    out[2] = 0.5 * p->kappa_c * h[1] * dV;
    double tot = out[1] + out[2];
    for (int k = 0; k < p->n_eta; ++k) { out[3 + k] = 0.5 * p->kappa_eta * h[2 + k] * dV; tot += out[3 + k]; }
    out[0] = tot;
    return PF_OK;
}

}  // namespace

extern "C" int pf_free_energy_static(const pf_params *p, const void *c, const void *eta, double *out)
{
    if (!p || !c || !out) return PF_EINVAL;
    if (p->ndim != 2 && p->ndim != 3) return PF_EINVAL;
    if (p->n_eta < 0 || p->n_eta > 8) return PF_EINVAL;
    if (p->n_eta > 0 && !eta) return PF_EINVAL;
    if (p->precision != PF_F32 && p->precision != PF_F64) return PF_EINVAL;
    long N = 1;
    for (int d = 0; d < p->ndim; ++d) {
        if (!(p->dx[d] > 0.0)) return PF_EINVAL;
        const int n = p->n[d];
        if (n < 16 || n > 2048 || (n & (n - 1))) return PF_EUNSUPPORTED;       // the grids pf_create accepts
        N *= n;
    }
    if (p->ndim == 2 && p->n[2] != 1) return PF_EUNSUPPORTED;
    if (N > (long)PF_STATIC_MAX_POINTS) return PF_EUNSUPPORTED;                // more tiles than the static array has slots for
    int ndev = 0, dev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev <= 0 || cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); return PF_ECUDA; }
    if (!device_readable(c, dev) || (p->n_eta > 0 && !device_readable(eta, dev))) return PF_EINVAL;
    double *scratch = nullptr;
    const int rc = scratch_of_current_device(&scratch);
    if (rc != PF_OK) return rc;
    return (p->precision == PF_F64) ? run<double>(p, c, eta, N, scratch, out) : run<float>(p, c, eta, N, scratch, out);
}
