// Host-side check of the exchange-buffer index map of the strided kernels (csrc/col_buf.cuh): for every shape the
// kernels instantiate, (1) load/store address every (row, slot) exactly once and agree with the reference map idx(),
// (2) the Stockham scatter followed by the gather moves each element to the register fft_core.cuh expects (checked
// through the data itself), (3) no shared-memory wavefront (128 consecutive bytes' worth of lanes) touches a bank twice.
// Built and run by tests/test_fft_core_host.py (no GPU needed). Exit code 0 = all pass.
#include <cstdio>
#include <set>
#include <vector>
#include "../../paper_2306_04322_b200/csrc/col_buf.cuh"

using namespace pf;

static int fails = 0, stages_checked = 0;

// records the element index of every access of one thread
template <typename C> struct Probe { long off; };

template <typename T, int N, int E, int TP, int NS> struct Stage {
    typedef typename V2<T>::type C;
    static constexpr int SLOTS = 2 * TP, TT = N / E, LR = (E >= 16) ? 4 : 3;
    typedef ColBuf<C, SLOTS, LR> Buf;
    static void go()
    {
        constexpr int R = stage_radix(N, E, NS);
        constexpr int LANES = 128 / (int)sizeof(C);
        std::vector<C> mem((size_t)N * SLOTS);
        // store phase: thread (sl, j) writes value encoding (destination row, slot)
        std::vector<std::vector<long>> st_addr(TT * SLOTS), ld_addr(TT * SLOTS);
        std::vector<int> hits((size_t)N * SLOTS, 0);
        for (int j = 0; j < TT; ++j)
            for (int sl = 0; sl < SLOTS; ++sl) {
                C v[E];
                constexpr int S = E / R;
                for (int m = 0; m < S; ++m) {
                    const int jv = j + m * TT, k = jv & (NS - 1), j0 = (jv - k) * R + k;
                    for (int r = 0; r < R; ++r) { v[m + r * S].x = (T)(j0 + r * NS); v[m + r * S].y = (T)sl; }
                }
                Buf b{mem.data(), sl};
                b.template store<N, E, NS>(v, j);
            }
        // every cell written exactly once with its own (row, slot) at the reference position
        for (int row = 0; row < N; ++row)
            for (int sl = 0; sl < SLOTS; ++sl) {
                const C c = mem[Buf::idx(row, sl)];
                if ((int)c.x != row || (int)c.y != sl) { if (fails < 5) printf("N=%d E=%d TP=%d NS=%d: cell (%d,%d) holds (%d,%d)\n", N, E, TP, NS, row, sl, (int)c.x, (int)c.y); ++fails; }
            }
        // gather: thread (sl, j) must receive rows j + q*TT of its slot
        for (int j = 0; j < TT; ++j)
            for (int sl = 0; sl < SLOTS; ++sl) {
                C v[E];
                Buf b{mem.data(), sl};
                b.template load<N, E>(v, j);
                for (int q = 0; q < E; ++q)
                    if ((int)v[q].x != j + q * TT || (int)v[q].y != sl) { ++fails; }
            }
        // bank conflicts: lanes are (slot fastest, then j); a wavefront = LANES consecutive lanes; within it all
        // element indices must fall into one 128-byte line or at least be distinct modulo the line size
        for (int j0 = 0; j0 + (LANES / SLOTS > 0 ? LANES / SLOTS : 1) <= TT; j0 += (LANES >= SLOTS ? LANES / SLOTS : 1)) {
            const int nj = LANES >= SLOTS ? LANES / SLOTS : 1;
            constexpr int S = E / R;
            for (int m = 0; m < S; ++m)
                for (int r = 0; r < R; ++r) {
                    std::set<int> pos;
                    int cnt = 0;
                    for (int dj = 0; dj < nj; ++dj)
                        for (int sl = 0; sl < (SLOTS < LANES ? SLOTS : LANES); ++sl) {
                            const int jv = j0 + dj + m * TT, k = jv & (NS - 1), jb = (jv - k) * R + k;
                            pos.insert(Buf::idx(jb + r * NS, sl) % LANES); ++cnt;
                        }
                    if ((int)pos.size() != cnt) { if (fails < 5) printf("N=%d E=%d TP=%d NS=%d: store bank conflict at j0=%d r=%d\n", N, E, TP, NS, j0, r); ++fails; }
                }
            for (int q = 0; q < E; ++q) {
                std::set<int> pos;
                int cnt = 0;
                for (int dj = 0; dj < nj; ++dj)
                    for (int sl = 0; sl < (SLOTS < LANES ? SLOTS : LANES); ++sl) { pos.insert(Buf::idx(j0 + dj + q * TT, sl) % LANES); ++cnt; }
                if ((int)pos.size() != cnt) { if (fails < 5) printf("N=%d E=%d TP=%d: load bank conflict at j0=%d q=%d\n", N, E, TP, j0, q); ++fails; }
            }
        }
        ++stages_checked;
        // the next exchange exists when the next stage is not the final one
        if constexpr (NS * R < N) {
            constexpr int NS2 = NS * R;
            if constexpr (NS2 * stage_radix(N, E, NS2) < N) Stage<T, N, E, TP, NS2>::go();
        }
    }
};

template <typename T, int N, int E, int TP> void shape()
{
    const int before = fails, s0 = stages_checked;
    if constexpr (stage_radix(N, E, 1) < N) Stage<T, N, E, TP, 1>::go();
    printf("%s N=%4d E=%2d TP=%d exchanges=%d %s\n", sizeof(T) == 8 ? "f64" : "f32", N, E, TP, stages_checked - s0, fails == before ? "ok" : "FAIL");
}

int main()
{
    shape<double, 16, 8, 8>(); shape<double, 32, 8, 8>(); shape<double, 64, 8, 4>(); shape<double, 128, 8, 4>();
    shape<double, 256, 8, 4>(); shape<double, 512, 8, 2>(); shape<double, 1024, 8, 2>(); shape<double, 2048, 8, 2>();
    shape<double, 2048, 8, 1>(); shape<double, 1024, 16, 2>();
    shape<float, 16, 8, 8>(); shape<float, 64, 8, 4>(); shape<float, 256, 8, 4>(); shape<float, 512, 8, 2>();
    shape<float, 1024, 8, 2>(); shape<float, 2048, 8, 2>(); shape<float, 2048, 8, 1>();
    shape<float, 1024, 16, 4>(); shape<float, 2048, 16, 2>(); shape<float, 2048, 16, 4>();
    if (fails) { printf("%d FAILURES\n", fails); return 1; }
    printf("ALL OK\n");
    return 0;
}
