// ttn_chimera.cuh -- Tropical<i16> sweep of the chimera-graph spin glass (
// PAPER.md:120-126, Fig. 2: M x N unit cells of K_{4,4}, "evolution of a state", Int16 elements).
//
// The paper contracts a network of 16 x 16 tropical matrices (one index per group of four spins).
// Here the same contraction runs at the level of single spins, in the circuit picture of
// every 16 x 16 inter-cell matrix is diagonal in the pairing of spin k with spin k,
// so it factorises into four 2 x 2 max-plus gates (A2) PAPER.md:242, and the intra-cell K_{4,4}
// tensor is a diagonal operator (a 256-entry table over the 4 + 4 spins of the cell).
//
// State: 2^(4M+4) int16 elements.  Index bits 0..3 = the ANCILLA: the vertical group v of the cell
// being processed (it is swept down the column); bits 4+4r .. 7+4r = the horizontal group u of row
// r (the boundary of the column sweep).  Bit = 0 means spin +1.  Two elements per 32-bit word
// (ancilla bit 0 = the half of a word), packed add / max / add-max instructions as in the
// Tropical<i16> Ising kernels.
//
// One launch = one cell (r, c) = one HBM pass over the state:
//   1. four gates on the bits of u^r with the couplings Jh[r][c-1][l] (u of column c-1 -> u of
//      column c; J = 0 in column 0: the state is still the tropical one there -- the very first
//      cell does not read it at all, it starts from zeros in registers);
//   2. four gates on the ancilla bits with Jv[r-1][c][k] (v of row r-1 -> v of row r; J = 0 for
//      r = 0, which maximises over the previous column's last v and broadcasts the result);
//   3. x += B(u, v) = sum_kl K[r][c][k][l] s_k(v) s_l(u), the cell's table.
// A thread owns the 256 elements that differ in the 8 active bits: 16 rows (u) of one 32-byte sector
// (v), 128 packed registers; consecutive threads own consecutive sectors of a row.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace ttn {

// One-warp CTAs: the warps of a CTA load, compute and store in phase, so what overlaps memory with
// the gates is CTAs of one SM being in different phases.  8 x 8 cells, per cell pass, one group per
// thread: 256 threads 89 ms, 128: 58.7, 64: 57.3, 32: 56.4 ms; capping the registers at 168 for
// 12 warps spills (69 - 81 ms).  With the grid-stride loop below (512 CTAs per SM): 48.7 ms.
// profiles/r01n.md.
#ifndef TTN_CH_THREADS
#define TTN_CH_THREADS 32
#endif
constexpr int CH_THREADS = TTN_CH_THREADS;
#ifndef TTN_CH_MINBLOCKS
#define TTN_CH_MINBLOCKS 1
#endif

struct ChimeraCellParams {
    unsigned* state;              // 2^(4M+3) words
    int p;                        // first bit of u^r in the ELEMENT index: 4 + 4 r
    int init;                     // the very first cell: the state is the tropical one (0), nothing is read
    unsigned long long groups;    // 2^(4M+4-8) threads' worth of work
    unsigned ju[4];               // packed (-2J, -2J) per spin l of u^r, as int16 pairs
    unsigned jv[4];               // packed (-2J, -2J) per spin k of the ancilla
    const unsigned* table;        // [16 u][8 words]: B(u, v), v = 2 j + half  (device)
};

// gate (A2) on a bit that selects between two packed words A (bit = 0) and B (bit = 1):
//   A' = max(A + J, B - J) = max(A, B - 2J) + J,  B' = max(B + J, A - 2J) = max(B, A - 2J) + J.
// The common + J is the same for every element of the state, so it is left out here and added to
// the final maximum on the host (sum of J over all gates): one VIADDMNMX per word and gate.
// m2 = packed (-2J, -2J).
__device__ __forceinline__ void ch_gate(unsigned& A, unsigned& B, const unsigned m2) {
    const unsigned na = __viaddmax_s16x2(B, m2, A);
    const unsigned nb = __viaddmax_s16x2(A, m2, B);
    A = na; B = nb;
}
// gate on the half of a word: w = (lo: bit = 0, hi: bit = 1)
__device__ __forceinline__ unsigned ch_gate_half(const unsigned w, const unsigned m2) {
    return __viaddmax_s16x2(__byte_perm(w, 0u, 0x1032), m2, w);
}

__global__ void __launch_bounds__(CH_THREADS, TTN_CH_MINBLOCKS) chimera_cell_kernel(const ChimeraCellParams q) {
    __shared__ uint4 s_tab[32];                       // 16 rows x 8 words
    if (threadIdx.x < 32) s_tab[threadIdx.x] = reinterpret_cast<const uint4*>(q.table)[threadIdx.x];
    __syncthreads();
    // a CTA walks the groups with the stride of the grid (ttn_api.cu sizes the grid)
    for (unsigned long long G = (unsigned long long)blockIdx.x * CH_THREADS + threadIdx.x; G < q.groups;
         G += (unsigned long long)gridDim.x * CH_THREADS) {
    // element index of (u = 0, v = 0): bits below p (above the ancilla) = low part of G, the rest above u^r
    const int midbits = q.p - 4;
    const unsigned long long mid = G & ((1ull << midbits) - 1), high = G >> midbits;
    const unsigned long long e0 = (mid << 4) + (high << (q.p + 4));
    uint4* base = reinterpret_cast<uint4*>(q.state + (e0 >> 1));
    const unsigned long long row_stride = (1ull << q.p) >> 3;       // uint4 (8 elements) per step of u
    unsigned w[16][8];
#pragma unroll
    for (int u = 0; u < 16; ++u) {
        const uint4 z = make_uint4(0u, 0u, 0u, 0u);                     // tropical one
        const uint4 a = q.init ? z : base[u * row_stride], b = q.init ? z : base[u * row_stride + 1];
        w[u][0] = a.x; w[u][1] = a.y; w[u][2] = a.z; w[u][3] = a.w;
        w[u][4] = b.x; w[u][5] = b.y; w[u][6] = b.z; w[u][7] = b.w;
    }
    // 1. gates on the four bits of u^r (row index)
#pragma unroll
    for (int l = 0; l < 4; ++l) {
        const unsigned m2 = q.ju[l];
#pragma unroll
        for (int u = 0; u < 16; ++u)
            if (!(u & (1 << l))) {
#pragma unroll
                for (int j = 0; j < 8; ++j) ch_gate(w[u][j], w[u | (1 << l)][j], m2);
            }
    }
    // 2. gates on the ancilla: bit 0 = the half, bits 1..3 = the word index
    {
        const unsigned m2 = q.jv[0];
#pragma unroll
        for (int u = 0; u < 16; ++u)
#pragma unroll
            for (int j = 0; j < 8; ++j) w[u][j] = ch_gate_half(w[u][j], m2);
    }
#pragma unroll
    for (int k = 1; k < 4; ++k) {
        const unsigned m2 = q.jv[k];
#pragma unroll
        for (int u = 0; u < 16; ++u)
#pragma unroll
            for (int j = 0; j < 8; ++j)
                if (!(j & (1 << (k - 1)))) ch_gate(w[u][j], w[u][j | (1 << (k - 1))], m2);
    }
    // 3. the cell's table, and store
#pragma unroll
    for (int u = 0; u < 16; ++u) {
        const uint4 ta = s_tab[2 * u], tb = s_tab[2 * u + 1];
        uint4 a, b;
        a.x = __vadd2(w[u][0], ta.x); a.y = __vadd2(w[u][1], ta.y); a.z = __vadd2(w[u][2], ta.z); a.w = __vadd2(w[u][3], ta.w);
        b.x = __vadd2(w[u][4], tb.x); b.y = __vadd2(w[u][5], tb.y); b.z = __vadd2(w[u][6], tb.z); b.w = __vadd2(w[u][7], tb.w);
        base[u * row_stride] = a; base[u * row_stride + 1] = b;
    }
    }
}

// The r = 0 cell of every column: u^0 sits next to the ancilla, so the 8 active bits are the 8 lowest
// index bits and a thread of the kernel above owns one contiguous 512 B (a warp's requests are then
// 512 B apart: 4.7 instead of 2.7 ms per pass at 7 x 7 cells).  Here a WARP owns 32 groups = 16 KiB
// contiguous and request i moves group i whole: lane L holds, of every group, the four words with
// u = L >> 1 and ancilla bit 3 = L & 1.  The gates on u and on ancilla bit 3 pair a word with the same
// word of another lane (the update max(w, partner - 2J) is the same on both sides: one SHFL.BFLY and
// one VIADDMNMX per word); ancilla bits 0..2 stay inside the thread.
__global__ void __launch_bounds__(CH_THREADS) chimera_cell0_kernel(const ChimeraCellParams q) {
    const int lane = threadIdx.x & 31;
    const uint4 tab = reinterpret_cast<const uint4*>(q.table)[lane];      // B(u = lane >> 1, v = 8 (lane & 1) + ...)
    const unsigned long long tiles = q.groups >> 5;                        // 32 groups each (host: groups >= 32)
    const unsigned long long warps = (unsigned long long)gridDim.x * (CH_THREADS / 32);
    for (unsigned long long T = (unsigned long long)blockIdx.x * (CH_THREADS / 32) + (threadIdx.x >> 5); T < tiles; T += warps) {
        uint4* base = reinterpret_cast<uint4*>(q.state) + (T << 10) + lane;   // 1024 uint4 per tile
        unsigned w[32][4];
#pragma unroll
        for (int i = 0; i < 32; ++i) {
            const uint4 a = q.init ? make_uint4(0u, 0u, 0u, 0u) : base[32 * i];
            w[i][0] = a.x; w[i][1] = a.y; w[i][2] = a.z; w[i][3] = a.w;
        }
        // gates on u^0 (lane bits 1..4) and on ancilla bit 3 (lane bit 0)
#pragma unroll
        for (int b = 0; b < 5; ++b) {
            const unsigned m2 = b == 0 ? q.jv[3] : q.ju[b - 1];
#pragma unroll
            for (int i = 0; i < 32; ++i)
#pragma unroll
                for (int j = 0; j < 4; ++j)
                    w[i][j] = __viaddmax_s16x2(__shfl_xor_sync(0xffffffffu, w[i][j], 1 << b), m2, w[i][j]);
        }
        // ancilla bit 0 (the half), bits 1, 2 (the word index inside the quad)
#pragma unroll
        for (int i = 0; i < 32; ++i) {
#pragma unroll
            for (int j = 0; j < 4; ++j) w[i][j] = ch_gate_half(w[i][j], q.jv[0]);
            ch_gate(w[i][0], w[i][1], q.jv[1]); ch_gate(w[i][2], w[i][3], q.jv[1]);
            ch_gate(w[i][0], w[i][2], q.jv[2]); ch_gate(w[i][1], w[i][3], q.jv[2]);
            base[32 * i] = make_uint4(__vadd2(w[i][0], tab.x), __vadd2(w[i][1], tab.y), __vadd2(w[i][2], tab.z), __vadd2(w[i][3], tab.w));
        }
    }
}

// max over the whole state (both halves of every word) -> *out (int, initialised to INT_MIN by the host side)
__global__ void __launch_bounds__(256) chimera_max_kernel(const uint4* __restrict__ state, const unsigned long long quads, int* out) {
    unsigned m2 = 0x80008000u;
    for (unsigned long long i = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; i < quads;
         i += (unsigned long long)gridDim.x * blockDim.x) {
        const uint4 t = state[i];
        m2 = __vmaxs2(__vmaxs2(m2, t.x), __vmaxs2(__vmaxs2(t.y, t.z), t.w));
    }
    int m = max((int)(short)(m2 & 0xffffu), (int)(short)(m2 >> 16));
    for (int o = 16; o; o >>= 1) m = max(m, __shfl_xor_sync(0xffffffffu, m, o));
    __shared__ int s[8];
    if ((threadIdx.x & 31) == 0) s[threadIdx.x >> 5] = m;
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int k = 1; k < 8; ++k) m = max(m, s[k]);
        atomicMax(out, m);
    }
}

}  // namespace ttn
