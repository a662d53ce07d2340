// dsmem_probe.cu -- pf_dsmem_read_rate (include/pf.h): how fast a CTA reads the shared memory of the OTHER CTAs of its
// thread-block cluster (distributed shared memory), in bytes per SM clock per SM, measured on the current device.
// Diagnostic only (like pf_fp64_fma_peak): the number decides SURVEY 8(f)-2's "merge the 3D y and z passes inside a
// cluster" -- every element of a plane would cross DSMEM once per transform direction -- and explains where the
// cluster-resident small-grid kernel (sgrid_kernels.cu) stops paying off (profiles/r3_dsmem.md).
//
// Kernel: one CTA per SM slot, clusters of `cs` CTAs, 512 threads, 32 KB of shared memory per CTA. After a cluster barrier
// every thread issues 16-byte loads (8 independent ones in flight) that walk the buffer of another CTA of the cluster --
// CTA (rank + 1 + k) mod cs for load k when `remote`, its own buffer through the same generic-address path otherwise --
// and the CTA's elapsed SM clocks are taken with clock64 around the loop. Rate = bytes the slowest CTA loaded / its clocks.
#include <cooperative_groups.h>
#include <cuda_runtime.h>

#include "../../include/pf.h"

namespace cg = cooperative_groups;

namespace {

constexpr int kThreads = 512;
constexpr int kVecs = 2048;                 // uint4 per CTA buffer: 32 KB
constexpr int kUnroll = 8;

__global__ void __launch_bounds__(kThreads) dsmem_probe_kernel(int iters, int remote, long long *cycles, unsigned *sink)
{
    __shared__ uint4 buf[kVecs];
    cg::cluster_group cluster = cg::this_cluster();
    const unsigned cs = cluster.num_blocks(), rank = cluster.block_rank();
    for (int i = threadIdx.x; i < kVecs; i += kThreads) buf[i] = make_uint4(i, rank, i ^ rank, 1u);
    cluster.sync();
    const uint4 *peer[kUnroll];
#pragma unroll
    for (int k = 0; k < kUnroll; ++k) peer[k] = cluster.map_shared_rank(buf, remote ? (rank + 1 + k % (cs > 1 ? cs - 1 : 1)) % cs : rank);
    unsigned acc = 0;
    __syncthreads();
    const long long t0 = clock64();
    int idx = threadIdx.x;
    for (int it = 0; it < iters; ++it) {
        uint4 v[kUnroll];
#pragma unroll
        for (int k = 0; k < kUnroll; ++k) v[k] = peer[k][(idx + k * kThreads) & (kVecs - 1)];
#pragma unroll
        for (int k = 0; k < kUnroll; ++k) acc ^= v[k].x + v[k].y + v[k].z + v[k].w;
        idx = (idx + 97) & (kVecs - 1);
    }
    __syncthreads();
    const long long t1 = clock64();
    if (threadIdx.x == 0) cycles[blockIdx.x] = t1 - t0;
    if (acc == 0x12345678u) sink[0] = acc;      // keeps the loads alive
    cluster.sync();                             // no CTA leaves while a neighbour still reads its buffer
}

}  // namespace

extern "C" int pf_dsmem_read_rate(int cluster_size, int remote, double *bytes_per_clk_per_sm)
{
    if (!bytes_per_clk_per_sm || cluster_size < 1 || cluster_size > 16 || (cluster_size & (cluster_size - 1))) return PF_EINVAL;
    auto kern = dsmem_probe_kernel;
    if (cluster_size > 8 && cudaFuncSetAttribute(kern, cudaFuncAttributeNonPortableClusterSizeAllowed, 1) != cudaSuccess) {
        cudaGetLastError();
        return PF_EUNSUPPORTED;
    }
    cudaLaunchConfig_t cfg = {};
    cfg.blockDim = dim3(kThreads);
    cfg.gridDim = dim3((unsigned)cluster_size);
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = (unsigned)cluster_size; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
    int nclusters = 0;
    if (cudaOccupancyMaxActiveClusters(&nclusters, kern, &cfg) != cudaSuccess) { cudaGetLastError(); return PF_ECUDA; }
    if (nclusters < 1) return PF_EUNSUPPORTED;
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) {
        cudaGetLastError();
        return PF_ECUDA;
    }
    // one CTA per SM: as many clusters as fit side by side, never more CTAs than SMs
    if (nclusters > sms / cluster_size) nclusters = sms / cluster_size;
    if (nclusters < 1) nclusters = 1;
    const int ctas = nclusters * cluster_size;
    cfg.gridDim = dim3((unsigned)ctas);
    long long *cycles = nullptr;
    unsigned *sink = nullptr;
    if (cudaMalloc((void **)&cycles, sizeof(long long) * ctas) != cudaSuccess || cudaMalloc((void **)&sink, 64) != cudaSuccess) {
        cudaGetLastError();
        if (cycles) cudaFree(cycles);
        return PF_ENOMEM;
    }
    const int iters = 4096;
    double best = 0.0;
    int rc = PF_OK;
    for (int rep = 0; rep < 3 && rc == PF_OK; ++rep) {           // first pass is the warm-up
        if (cudaLaunchKernelEx(&cfg, kern, iters, remote, cycles, sink) != cudaSuccess || cudaDeviceSynchronize() != cudaSuccess) {
            cudaGetLastError();
            rc = PF_ECUDA;
            break;
        }
        long long h[160];
        if (cudaMemcpy(h, cycles, sizeof(long long) * (ctas < 160 ? ctas : 160), cudaMemcpyDeviceToHost) != cudaSuccess) { rc = PF_ECUDA; break; }
        long long worst = 1;
        for (int i = 0; i < ctas && i < 160; ++i) if (h[i] > worst) worst = h[i];
        const double rate = (double)iters * kUnroll * kThreads * 16.0 / (double)worst;
        if (rep > 0 && rate > best) best = rate;
    }
    cudaFree(cycles); cudaFree(sink);
    *bytes_per_clk_per_sm = best;
    return rc;
}
