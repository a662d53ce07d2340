// Host-side emulation of the thread-cooperative Stockham FFT in csrc/fft_core.cuh: the per-thread
// stage/exchange functions are run for every emulated thread, phase by phase (a phase boundary is where
// the kernels place a barrier), and the result is compared with a naive long-double DFT written here.
// Built and run by tests/test_fft_core_host.py (no GPU needed). Exit code 0 = all sizes pass.
#include <cmath>
#include <cstdio>
#include <vector>
#include "../../paper_2306_04322_b200/csrc/fft_core.cuh"

using namespace pf;

template <typename C> struct HostBuf {
    std::vector<C> *d;
    __host__ __device__ void st(int i, C v) { (*d)[i] = v; }
    __host__ __device__ C ld(int i) const { return (*d)[i]; }
};

template <typename T, int N, int E, int NS> struct Run {
    typedef typename V2<T>::type C;
    static void go(std::vector<std::vector<C>> &regs, const std::vector<C> &tw)
    {
        constexpr int TT = N / E;
        constexpr int R = stage_radix(N, E, NS);
        for (int j = 0; j < TT; ++j) { C (&v)[E] = *reinterpret_cast<C (*)[E]>(regs[j].data()); stage_compute<N, E, NS>(v, j, tw.data()); }
        if constexpr (NS * R < N) {
            std::vector<C> smem(N);
            HostBuf<C> buf{&smem};
            for (int j = 0; j < TT; ++j) { C (&v)[E] = *reinterpret_cast<C (*)[E]>(regs[j].data()); exchange_store<N, E, NS>(v, j, buf); }
            for (int j = 0; j < TT; ++j) { C (&v)[E] = *reinterpret_cast<C (*)[E]>(regs[j].data()); exchange_load<N, E>(v, j, buf); }
            Run<T, N, E, NS * R>::go(regs, tw);
        }
    }
};

template <typename T, int N, int E> double check()
{
    typedef typename V2<T>::type C;
    constexpr int TT = N / E;
    const long double PI = 3.141592653589793238462643383279502884L;
    std::vector<C> tw(N);
    for (int i = 0; i < N; ++i) { tw[i].x = (T)cosl(2 * PI * i / N); tw[i].y = (T)-sinl(2 * PI * i / N); }
    std::vector<long double> xr(N), xi(N);
    unsigned s = 12345u + N * 7 + E;
    for (int i = 0; i < N; ++i) {
        s = s * 1664525u + 1013904223u; xr[i] = (long double)(s >> 8) / (1 << 24) - 0.5L;
        s = s * 1664525u + 1013904223u; xi[i] = (long double)(s >> 8) / (1 << 24) - 0.5L;
    }
    std::vector<std::vector<C>> regs(TT, std::vector<C>(E));
    for (int j = 0; j < TT; ++j) for (int q = 0; q < E; ++q) { regs[j][q].x = (T)xr[j + q * TT]; regs[j][q].y = (T)xi[j + q * TT]; }
    Run<T, N, E, 1>::go(regs, tw);
    double err = 0, nrm = 0;
    for (int k = 0; k < N; ++k) {
        long double sr = 0, si = 0;
        for (int n = 0; n < N; ++n) {
            long double a = -2 * PI * (long double)((long)n * k % N) / N;
            // use the rounded inputs the transform actually saw
            long double ur = (long double)(T)xr[n], ui = (long double)(T)xi[n];
            sr += ur * cosl(a) - ui * sinl(a); si += ur * sinl(a) + ui * cosl(a);
        }
        const C got = regs[k % TT][k / TT];
        err = fmax(err, fmax(fabs((double)(got.x - sr)), fabs((double)(got.y - si))));
        nrm = fmax(nrm, fmax(fabs((double)sr), fabs((double)si)));
    }
    return err / nrm;
}

static int fails = 0;
template <typename T, int N, int E> void one(double tol)
{
    double e = check<T, N, E>();
    printf("%s N=%4d E=%2d stages=%d rel_err=%.3e %s\n", sizeof(T) == 8 ? "f64" : "f32", N, E, num_stages(N, E), e, e < tol ? "ok" : "FAIL");
    if (!(e < tol)) ++fails;
}

int main()
{
    // radix-R butterflies alone (single thread, N = E)
    one<double, 2, 2>(1e-15); one<double, 4, 4>(1e-15); one<double, 8, 8>(1e-15); one<double, 16, 16>(1e-15); one<double, 32, 32>(2e-15);
    one<double, 8, 4>(1e-15); one<double, 16, 8>(1e-15); one<double, 32, 8>(1e-15); one<double, 64, 8>(1e-15);
    one<double, 128, 8>(2e-15); one<double, 256, 8>(2e-15); one<double, 512, 8>(2e-15); one<double, 1024, 8>(2e-15); one<double, 2048, 8>(3e-15);
    one<double, 16, 16>(1e-15); one<double, 64, 16>(1e-15); one<double, 256, 16>(2e-15); one<double, 512, 16>(2e-15);
    one<double, 1024, 16>(2e-15); one<double, 2048, 16>(3e-15); one<double, 1024, 32>(2e-15); one<double, 512, 32>(2e-15);
    one<double, 64, 4>(1e-15); one<double, 256, 4>(2e-15);
    one<float, 64, 8>(1e-6); one<float, 512, 8>(2e-6); one<float, 1024, 8>(2e-6); one<float, 2048, 16>(2e-6); one<float, 256, 16>(1e-6);
    printf(fails ? "FAILED %d\n" : "ALL OK\n", fails);
    return fails ? 1 : 0;
}
