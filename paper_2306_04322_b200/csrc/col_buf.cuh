// col_buf.cuh -- shared-memory exchange buffer of the strided-direction kernels (product code; shares nothing with
// oracle/). __host__ __device__ so that tests/test_fft_core_host.py can check the index map on the CPU.
//
// The buffer holds N rows (index along the FFT axis) of SLOTS column slots, one complex each. A shared-memory
// wavefront serves 128 bytes = LANES consecutive lanes; lanes are ordered (slot fastest, then the row-group index j),
// so a wavefront covers L = LANES/SLOTS different rows of all SLOTS columns. Which rows depends on the access:
//   loads (rows j + q*TT, consecutive j) and stores of the later stages: rows that differ in their low log2(L) bits;
//   stores of the first stage (rows R*j + r):                             rows that differ in bits [LR, LR + log2 L).
// Rows are therefore placed at  line = row / L,  position in line = (row ^ (row >> LR)) mod L,  which is distinct
// within a wavefront under both patterns (no bank conflicts) and is XOR-linear in the row index, so that the
// offsets of the E accesses of a thread differ from a per-thread base by compile-time constants.
#pragma once
#include "fft_core.cuh"

namespace pf {

template <typename C, int SLOTS, int LR> struct ColBuf {
    static constexpr int LANES = 128 / (int)sizeof(C);
    static constexpr int L = (SLOTS >= LANES) ? 1 : LANES / SLOTS;        // rows per 128-byte line
    C *base;
    int slot;

    PF_HD static constexpr int sub(int row) { return (row ^ (row >> LR)) & (L - 1); }
    // element index of (row, slot): reference form of the map
    PF_HD static constexpr int idx(int row, int slot) { return ((row & ~(L - 1)) + sub(row)) * SLOTS + slot; }

    // v[q] <- row j + q*TT
    template <int N, int E> PF_HD void load(C (&v)[E], int j) const
    {
        constexpr int TT = N / E;
        static_assert(TT >= L || L == 1, "row groups smaller than a line");
        int b[L];
        const int hi = (j & ~(L - 1)) * SLOTS + slot, sj = sub(j);
#pragma unroll
        for (int c = 0; c < L; ++c) b[c] = hi + (sj ^ c) * SLOTS;
#pragma unroll
        for (int q = 0; q < E; ++q) v[q] = base[b[sub(q * TT)] + ((q * TT) & ~(L - 1)) * SLOTS];
    }

    // Stockham scatter of the stage that starts at NS (fft_core.cuh): element r of butterfly jv -> row (jv-k)*R + k + r*NS
    template <int N, int E, int NS> PF_HD void store(const C (&v)[E], int j)
    {
        constexpr int R = stage_radix(N, E, NS);
        constexpr int S = E / R;
        constexpr int TT = N / E;
#pragma unroll
        for (int m = 0; m < S; ++m) {
            const int jv = j + m * TT;
            const int k = jv & (NS - 1);
            const int j0 = (jv - k) * R + k;
            int b[L];
            const int hi = (j0 & ~(L - 1)) * SLOTS + slot, s0 = sub(j0);
#pragma unroll
            for (int c = 0; c < L; ++c) b[c] = hi + (s0 ^ c) * SLOTS;
#pragma unroll
            for (int r = 0; r < R; ++r) base[b[sub(r * NS)] + ((r * NS) & ~(L - 1)) * SLOTS] = v[m + r * S];
        }
    }
};

}  // namespace pf
