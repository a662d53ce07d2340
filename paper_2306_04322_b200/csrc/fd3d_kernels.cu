// fd3d_kernels.cu -- the explicit forward-Euler finite-difference step in 3D,
// 7-point Laplacian, periodic wrap, every right-hand side at time t, ONE launch per step:
//     mu = df/dc - kappa_c lap c,   c' = c + dt M lap mu,   eta_i' = eta_i - dt L (df/deta_i - kappa_eta lap eta_i).
//
// A CTA owns a 64 x 8 tile of (x, y) and marches along a chunk of z. Every thread owns TWO neighbouring x points of
// one tile row, so shared-memory reads, global stores and the cp.async tile loads all move pairs (16 bytes in fp64).
// Shared memory holds rings of planes: c with a halo of two points (four slots), every eta_i with a halo of one (four
// slots) and mu on the tile plus a ring of one point (three slots). The z neighbours of a thread's own points --
// c(k..k+2), mu(k-1..k+1), eta(k-1..k+1) -- live in registers and march with k. Iteration k, ONE barrier:
//     wait for c(k+3), eta(k+2); barrier; queue c(k+4), eta(k+3) (cp.async, lands during the iteration)
//     mu(k+2) on the tile and its ring   (reads c(k+1..k+3), eta(k+2); writes the third mu slot)
//     c', eta_i' of plane k               (reads mu(k), eta(k) x-y neighbours from shared memory, the rest from registers)
// The two halves do not depend on each other, so every thread carries two instruction streams and nothing waits for a
// second barrier (the two-barrier form of this kernel ran 256^3, c + 2 eta, in 293 us, this one in 204 us;
// fd_fused3d_kernel in fd_kernels.cu, one point per thread, in 348 us; profiles/r2_fd3d.md).
// The ring of mu is dealt out warp by warp: the two extra rows to warps 0 and 1 (same pair code as the tile rows), the
// two extra columns to one warp, so no warp runs a pass with two active lanes.
// Up to four order parameters (126 registers, two CTAs per SM); more run fd_fused3d_kernel.
#include <atomic>
#include "pf_kernels.cuh"

namespace pf {

namespace {

template <typename T> struct Pair;
template <> struct Pair<double> { typedef double2 type; };
template <> struct Pair<float>  { typedef float2  type; };

// global -> shared copy of one pair of points without a register stop-over
template <typename T> __device__ __forceinline__ void cp_async_pair(T *smem_dst, const T *gmem_src)
{
    asm volatile("cp.async.ca.shared.global [%0], [%1], %2;" ::"r"((unsigned)__cvta_generic_to_shared(smem_dst)), "l"(gmem_src), "n"(2 * sizeof(T)) : "memory");
}
__device__ __forceinline__ void cp_async_wait_all_pairs() { asm volatile("cp.async.wait_all;" ::: "memory"); }

__device__ __forceinline__ int wrap_inc(int i, int n) { return (i + 1 == n) ? 0 : i + 1; }

}  // namespace

template <typename T, int NE>
__global__ void __launch_bounds__(256, 2) fd3d_march_kernel(const FdParams<T> p, const int zc)
{
    typedef typename Pair<T>::type P2;
    constexpr int TX = 64, TY = 8, PW = TX + 4;          // pitch of every plane in shared memory (x halo of two points)
    constexpr int CH = TY + 4, EH = TY + 2;              // rows of a c plane / of an eta or mu plane
    constexpr int CP = CH * PW, EP = EH * PW;
    constexpr int CS = 4, ES = 4, MS = 3;                // ring slots
    constexpr int NC = (CP / 2 + 255) / 256, NEC = (EP / 2 + 255) / 256;   // pair copies per thread and plane
    extern __shared__ __align__(16) unsigned char fd3_smem[];
    T *sc = reinterpret_cast<T *>(fd3_smem);             // [CS][CP]
    T *smu = sc + CS * CP;                               // [MS][EP]
    T *se = smu + MS * EP;                               // [NE][ES][EP]

    const int tid = threadIdx.x;
    const int tx = tid & 31, ty = tid >> 5;              // one warp per tile row
    const int x0 = blockIdx.x * TX, y0 = blockIdx.y * TY;
    const int z0 = blockIdx.z * zc;
    const int zn = min(zc, p.nz - z0);                   // planes of this chunk
    const int mx = p.nx - 1, my = p.ny - 1, mz = p.nz - 1;
    const long plane = (long)p.nx * p.ny;
    const T rx = p.rdx2[0], ry = p.rdx2[1], rz = p.rdx2[2];

    // per-thread copy lists (the same for every plane): shared-memory offset and wrapped global offset of each pair
    int cs_off[NC], cg_off[NC], es_off[NEC], eg_off[NEC];
#pragma unroll
    for (int i = 0; i < NC; ++i) {
        const int t = tid + i * 256;
        const int row = t / (PW / 2), cp = t - row * (PW / 2);
        cs_off[i] = (t < CP / 2) ? row * PW + 2 * cp : -1;
        cg_off[i] = ((y0 + row - 2) & my) * p.nx + ((x0 + 2 * cp - 2) & mx);
    }
#pragma unroll
    for (int i = 0; i < NEC; ++i) {
        const int t = tid + i * 256;
        const int row = t / (PW / 2), cp = t - row * (PW / 2);
        es_off[i] = (t < EP / 2) ? row * PW + 2 * cp : -1;
        eg_off[i] = ((y0 + row - 1) & my) * p.nx + ((x0 + 2 * cp - 2) & mx);
    }
    auto load_c = [&](int m, int slot) {                 // plane z0 + m
        const T *src = p.c + (long)((z0 + m) & mz) * plane;
        T *dst = sc + slot * CP;
#pragma unroll
        for (int i = 0; i < NC; ++i)
            if (cs_off[i] >= 0) cp_async_pair(dst + cs_off[i], src + cg_off[i]);
    };
    auto load_e = [&](int m, int slot) {
#pragma unroll
        for (int f = 0; f < NE; ++f) {
            const T *src = p.eta + (long)f * p.fs + (long)((z0 + m) & mz) * plane;
            T *dst = se + (f * ES + slot) * EP;
#pragma unroll
            for (int i = 0; i < NEC; ++i)
                if (es_off[i] >= 0) cp_async_pair(dst + es_off[i], src + eg_off[i]);
        }
    };

    // offsets of this thread's two points: column ix = 2 + 2 tx of row ty + 2 (c planes) / ty + 1 (eta, mu planes)
    const int ix = 2 + 2 * tx;
    const int own_c = (ty + 2) * PW + ix, own_e = (ty + 1) * PW + ix;
    auto ld2 = [](const T *q) { return *reinterpret_cast<const P2 *>(q); };

    // x-y part of the Laplacian of a pair at offset o of plane P (centre pair v given)
    auto lap_xy = [&](const T *P, int o, P2 v) {
        const T l = P[o - 1], r = P[o + 2];
        const P2 u = ld2(P + o - PW), d = ld2(P + o + PW);
        P2 out;
        out.x = rx * (l + v.y - T(2) * v.x) + ry * (u.x + d.x - T(2) * v.x);
        out.y = rx * (v.x + r - T(2) * v.y) + ry * (u.y + d.y - T(2) * v.y);
        return out;
    };
    // kernel (i) for a pair: mu = df/dc - kappa_c lap c. oc / oe: offsets in a c plane / an eta plane;
    // c0 = plane of the pair, vm / vp = the pair one plane below / above, eslot = slot of the eta plane
    auto mu_pair = [&](const T *c0, int oc, P2 v, P2 vm, P2 vp, int eslot, int oe, const P2 *eown) {
        P2 l = lap_xy(c0, oc, v);
        l.x += rz * (vm.x + vp.x - T(2) * v.x);
        l.y += rz * (vm.y + vp.y - T(2) * v.y);
        T h0 = 0, h1 = 0;
#pragma unroll
        for (int f = 0; f < NE; ++f) {
            const P2 e = eown ? eown[f] : ld2(se + (f * ES + eslot) * EP + oe);
            h0 += h_term(e.x); h1 += h_term(e.y);
        }
        P2 mu;
        mu.x = dfdc(p.m, v.x, h0) - p.m.kappa_c * l.x;
        mu.y = dfdc(p.m, v.y, h1) - p.m.kappa_c * l.y;
        return mu;
    };
    // the ring of mu(m): rows -1 and TY (warps 0, 1: pairs) and columns -1 and TX (warp 2: single points).
    // cslot = slot of c(m), cm / cp its neighbours, eslot = slot of eta(m), mslot = slot of mu(m)
    auto mu_ring = [&](int cslot, int cmslot, int cpslot, int eslot, int mslot) {
        const T *c0 = sc + cslot * CP, *cm = sc + cmslot * CP, *cp = sc + cpslot * CP;
        T *mu = smu + mslot * EP;
        if (ty < 2) {
            const int rr = ty ? TY + 1 : 0;                               // mu row (y0 - 1 or y0 + TY)
            const int oc = (rr + 1) * PW + ix, oe = rr * PW + ix;
            const P2 v = ld2(c0 + oc);
            const P2 m2 = mu_pair(c0, oc, v, ld2(cm + oc), ld2(cp + oc), eslot, oe, nullptr);
            *reinterpret_cast<P2 *>(mu + oe) = m2;
        } else if (ty == 2 && tx < 2 * EH) {
            const int rr = tx >> 1, col = (tx & 1) ? TX + 2 : 1;
            const int oc = (rr + 1) * PW + col, oe = rr * PW + col;
            const T v = c0[oc];
            const T l = rx * (c0[oc - 1] + c0[oc + 1] - T(2) * v) + ry * (c0[oc - PW] + c0[oc + PW] - T(2) * v)
                      + rz * (cm[oc] + cp[oc] - T(2) * v);
            T h = 0;
#pragma unroll
            for (int f = 0; f < NE; ++f) h += h_term(se[(f * ES + eslot) * EP + oe]);
            mu[oe] = dfdc(p.m, v, h) - p.m.kappa_c * l;
        }
    };

    grid_dependency_wait();
    grid_dependents_launch();

    const long g0 = (long)(y0 + ty) * p.nx + (x0 + 2 * tx);
    // kernels (ii) + (iii) for this thread's pair of plane zk: mu and eta planes of that z in slots ms / es (x-y
    // neighbours), z neighbours from registers
    auto update_pair = [&](int zk, int ms, int es, P2 ck, P2 mum, P2 mu0, P2 mup, const P2 *em, const P2 *e0, const P2 *ep) {
        const long g = (long)((z0 + zk) & mz) * plane + g0;
        {
            P2 lm = lap_xy(smu + ms * EP, own_e, mu0);
            lm.x += rz * (mum.x + mup.x - T(2) * mu0.x);
            lm.y += rz * (mum.y + mup.y - T(2) * mu0.y);
            P2 cn; cn.x = ck.x + p.m.dtM * lm.x; cn.y = ck.y + p.m.dtM * lm.y;
            *reinterpret_cast<P2 *>(p.c_new + g) = cn;
        }
        T s0 = 0, s1 = 0;
#pragma unroll
        for (int f = 0; f < NE; ++f) { s0 += e0[f].x * e0[f].x; s1 += e0[f].y * e0[f].y; }
#pragma unroll
        for (int f = 0; f < NE; ++f) {
            P2 le = lap_xy(se + (f * ES + es) * EP, own_e, e0[f]);
            le.x += rz * (em[f].x + ep[f].x - T(2) * e0[f].x);
            le.y += rz * (em[f].y + ep[f].y - T(2) * e0[f].y);
            P2 en;
            en.x = e0[f].x - p.m.dtL * (dfdeta(p.m, ck.x, e0[f].x, s0) - p.m.kappa_eta * le.x);
            en.y = e0[f].y - p.m.dtL * (dfdeta(p.m, ck.y, e0[f].y, s1) - p.m.kappa_eta * le.y);
            *reinterpret_cast<P2 *>(p.eta_new + (long)f * p.fs + g) = en;
        }
    };

    {
        // One barrier per plane: iteration k forms mu(k+2) and, independently of it, c', eta' of plane k from mu(k-1..k+1)
        // of earlier iterations -- two instruction streams per thread and no barrier between them.
        // slots: c(m) in (m + 4) mod 4, eta(m) in (m + 4) mod 4, mu(m) in m mod 3
        constexpr int NR = NE > 0 ? NE : 1;
        load_c(-2, 2); load_c(-1, 3); load_c(0, 0); load_c(1, 1);
        load_e(-1, 3); load_e(0, 0); load_e(1, 1);
        cp_async_wait_all_pairs();
        __syncthreads();
        P2 ck, c1, c2, mum, mu0, mup;                     // own points: c(k..k+2), mu(k-1..k+1)
        P2 em[NR], e0[NR], ep[NR];                        // eta(k-1..k+1)
        {
            const P2 cm1 = ld2(sc + 3 * CP + own_c);
            ck = ld2(sc + 0 * CP + own_c);
            c1 = ld2(sc + 1 * CP + own_c);
#pragma unroll
            for (int f = 0; f < NE; ++f) {
                em[f] = ld2(se + (f * ES + 3) * EP + own_e); e0[f] = ld2(se + (f * ES + 0) * EP + own_e);
                ep[f] = ld2(se + (f * ES + 1) * EP + own_e);
            }
            mum = mu_pair(sc + 3 * CP, own_c, cm1, ld2(sc + 2 * CP + own_c), ck, 3, own_e, NE > 0 ? em : nullptr);   // own points only
            mu0 = mu_pair(sc + 0 * CP, own_c, ck, cm1, c1, 0, own_e, NE > 0 ? e0 : nullptr);
            *reinterpret_cast<P2 *>(smu + 0 * EP + own_e) = mu0;
            mu_ring(0, 3, 1, 0, 0);
        }
        __syncthreads();                                  // c(-2) is dead
        load_c(2, 2); load_e(2, 2);
        cp_async_wait_all_pairs();
        __syncthreads();
        c2 = ld2(sc + 2 * CP + own_c);
        mup = mu_pair(sc + 1 * CP, own_c, c1, ck, c2, 1, own_e, NE > 0 ? ep : nullptr);
        *reinterpret_cast<P2 *>(smu + 1 * EP + own_e) = mup;
        mu_ring(1, 0, 2, 1, 1);
        load_c(3, 3);                                     // slot of c(-1): dead since the barrier above

        int cs = 0, ms = 0;                               // slots of c(k) (= slot of eta(k)) and of mu(k)
        for (int k = 0; k < zn; ++k) {
            cp_async_wait_all_pairs();
            __syncthreads();                              // c(k+3), eta(k+2) have landed; mu(k+1) is complete
            const int cs1 = (cs + 1) & 3, cs2 = (cs + 2) & 3, cs3 = (cs + 3) & 3;
            const int ms1 = wrap_inc(ms, MS), ms2 = wrap_inc(ms1, MS);
            if (k + 1 < zn) { load_c(k + 4, cs); load_e(k + 3, cs3); }     // over c(k) and eta(k-1): registers hold what is needed

            // mu(k+2): own pair, then the ring
            const P2 c3 = ld2(sc + cs3 * CP + own_c);
            P2 e2[NR];
#pragma unroll
            for (int f = 0; f < NE; ++f) e2[f] = ld2(se + (f * ES + cs2) * EP + own_e);
            const P2 mu2 = mu_pair(sc + cs2 * CP, own_c, c2, c1, c3, cs2, own_e, NE > 0 ? e2 : nullptr);
            *reinterpret_cast<P2 *>(smu + ms2 * EP + own_e) = mu2;
            update_pair(k, ms, cs, ck, mum, mu0, mup, em, e0, ep);
            mu_ring(cs2, cs1, cs3, cs2, ms2);
            // march
            ck = c1; c1 = c2; c2 = c3; mum = mu0; mu0 = mup; mup = mu2;
#pragma unroll
            for (int f = 0; f < NE; ++f) { em[f] = e0[f]; e0[f] = ep[f]; ep[f] = e2[f]; }
            cs = cs1; ms = ms1;
        }
    }
}

template <typename T, int NE> static cudaError_t launch_fd3d_march_ne(const FdParams<T> &p, cudaStream_t s)
{
    constexpr int TX = 64, TY = 8, PW = TX + 4, CP = (TY + 4) * PW, EP = (TY + 2) * PW;
    constexpr int ES = 4, MS = 3;
    const size_t smem = sizeof(T) * ((size_t)4 * CP + (size_t)(MS + ES * NE) * EP);
    auto kern = fd3d_march_kernel<T, NE>;
    // Function attributes and occupancy belong to a DEVICE: a process may hold contexts on several (pf.h), so both are
    // looked up once per device (index = CUDA device ordinal), not once per process.
    constexpr int MAXDEV = 64;
    static std::atomic<int> per_sm_of[MAXDEV];           // resident CTAs per SM of this instantiation; 0 = not yet set up
    int dev = 0, sms = 148;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= MAXDEV) return cudaErrorInvalidDevice;
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    int per_sm = per_sm_of[dev].load(std::memory_order_acquire);
    if (per_sm == 0) {
        if ((e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem)) != cudaSuccess) return e;
        int n = 0;
        if ((e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, kern, 256, smem)) != cudaSuccess) return e;
        per_sm = n > 0 ? n : 1;
        per_sm_of[dev].store(per_sm, std::memory_order_release);     // two threads racing here store the same value
    }
    // chunks along z: every chunk re-reads four planes, and the CTAs should fill whole waves. Pick the chunk count with
    // the best (fill of the last wave) x (useful planes / planes read).
    const int tiles = (p.nx / TX) * (p.ny / TY);
    const double slots = (double)sms * per_sm;
    int best = 1; double best_eff = -1.0;
    for (int ch = 1; ch <= p.nz / 8 || ch == 1; ++ch) {
        const int zc = (p.nz + ch - 1) / ch;
        const int used = (p.nz + zc - 1) / zc;
        if (used != ch) continue;
        const double waves = tiles * (double)ch / slots;
        const double eff = waves / (double)(long)(waves + 0.999999) * zc / (zc + 5.0);
        if (eff > best_eff) { best_eff = eff; best = ch; }
    }
    const int zc = (p.nz + best - 1) / best;
    return launch_pdl(kern, dim3((unsigned)(p.nx / TX), (unsigned)(p.ny / TY), (unsigned)best), dim3(256), smem, s, true, p, zc);
}

// nx >= 64, ny >= 8 (both powers of two). Other shapes: fd_fused3d_kernel (fd_kernels.cu).
template <typename T> cudaError_t launch_fd3d_march(const FdParams<T> &p, cudaStream_t s)
{
    if (p.nx < 64 || p.ny < 8) return cudaErrorNotSupported;
    switch (p.m.n_eta) {
    case 0: return launch_fd3d_march_ne<T, 0>(p, s);
    case 1: return launch_fd3d_march_ne<T, 1>(p, s);
    case 2: return launch_fd3d_march_ne<T, 2>(p, s);
    case 3: return launch_fd3d_march_ne<T, 3>(p, s);
    case 4: return launch_fd3d_march_ne<T, 4>(p, s);
    }
    return cudaErrorNotSupported;
}

template cudaError_t launch_fd3d_march<double>(const FdParams<double> &, cudaStream_t);
template cudaError_t launch_fd3d_march<float>(const FdParams<float> &, cudaStream_t);

}  // namespace pf
