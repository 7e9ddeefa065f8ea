// ttn_chimera2.cuh -- chimera-graph spin glass on the paper's own state: "evolution of a state with
// dimension 16^L", Tropical<i16>, one index of dimension 16 per HORIZONTAL group of
// four spins and NO ancilla in HBM (ttn_chimera.cuh keeps a 4-spin ancilla in the state: 16 x the
// bytes; it stays as the path for M <= 3 rows of cells, where this one has too few bits to tile).
//
// State F[u], u = (u^0 .. u^{M-1}), bit 4 r + l = spin l of the horizontal group of row r (0 = up),
// 2^(4M) int16 elements, two per 32-bit word (bit 0 = the half).  Column c of the M x N cells:
//   1. (c >= 1) the 4 M inter-cell couplings Jh[r][c-1][l] are single-spin max-plus gates (A2)
//      PAPER.md:242 on the bits of u: they run on the Tropical<i16> Ising pass kernels (ttn_fused.cuh)
//      as ONE gate row of a 4M-column lattice whose row diagonals are zero;
//   2. the column's vertical chain -- the cells' K_{4,4} tensors B_r(u^r, v^r) and the 16 x 16 matrices
//      of the vertical couplings Jv[r-1][c] between v^{r-1} and v^r (Fig. 2b) --
//      contracts, for fixed u, to a number G_c(u): a diagonal operator on the state,
//          F[u] += G_c(u),   G_c(u) = max_{v^0..v^{M-1}} sum_r B_r(u^r, v^r) + sum_r V_{r-1}(v^{r-1}, v^r).
//      chimera_column_kernel below evaluates G_c(u) on the fly, from the TOP row down, so that what the
//      elements of a tile share is computed once per tile:
//          a_r[v] = B_r(u^r, v) + b_{r+1}[v],   b_r[v] = max_{v'} ( a_r[v'] + V_{r-1}(v, v') ),   G = max_v a_0[v],
//      with 16-entry vectors of int16 (8 packed words); V is four single-spin gates (one VIADDMNMX.S16x2
//      per word and gate, the common + J deferred to the host as everywhere).
// (The gate on the TOP bit of u is not part of the gate-row passes: the column kernel applies it to
// the pair of tiles that differ in that bit, in front of the diagonal -- one pass less per column.)
// A warp owns a tile of 2^12 elements (u^0, u^1, u^2; 8 KiB contiguous): lane = (bit 3 of u^0, u^1),
// a lane's 16 uint4 = the 16 values of u^2 x the 8 low values of u^0.  Levels r >= 3 are uniform
// per tile; level 2 runs once per u^2, level 1 once per (u^2, lane), level 0 is a 16-term add-max per
// element against the lane's rows of B_0 held in registers.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>
#include "ttn_chimera.cuh"

namespace ttn {

constexpr int CH2_WARPS = 8;

struct ChimeraColumnParams {
    unsigned* state;              // 2^(4M-1) words
    int M;                        // rows of cells, 4 <= M <= 8
    int init;                     // column 0: the state is the tropical one (0): nothing is read
    int reduce;                   // last column: nothing is stored; max_u F[u] -> atomicMax(out)
    unsigned long long tiles;     // 2^(4M-12)
    const unsigned* tables;       // [M rows][16 u][8 words]: B_r(u, v) of this column, v = 2 j + half
    unsigned jv[8][4];            // [r][k] packed (-2J, -2J) of Jv[r-1][c][k]; row 0 unused
    unsigned ju_top;              // packed (-2J, -2J) of the horizontal coupling on the top bit of u (0 in column 0)
    int* out;
};

// b[v] = max_{v'} (a[v'] + V(v, v')) up to the deferred constant: the four single-spin gates of the
// 16 x 16 matrix of one vertical coupling group.  Word j holds v = 2 j (lo), 2 j + 1 (hi).
__device__ __forceinline__ void ch2_vgates(unsigned (&x)[8], const unsigned (&m2)[4]) {
#pragma unroll
    for (int j = 0; j < 8; ++j) x[j] = ch_gate_half(x[j], m2[0]);
#pragma unroll
    for (int k = 1; k < 4; ++k) {
        const int B = 1 << (k - 1);
#pragma unroll
        for (int j = 0; j < 8; ++j)
            if (!(j & B)) ch_gate(x[j], x[j | B], m2[k]);
    }
}

// One element block of the column update: G(u) for the lane's uint4 of tile `tile` at u^2 = i, given b_3.
__device__ __forceinline__ uint4 ch2_column_G(const unsigned (&b3)[8], const int i, const uint4 (*s_tab)[32],
                                              const unsigned (&T0)[8][8], const unsigned (&T1)[8],
                                              const unsigned (&jv1)[4], const unsigned (&jv2)[4]) {
    // ---- level 2 (uniform per warp), level 1 (per lane)
    unsigned x[8];
    {
        const uint4 lo = s_tab[2][2 * i], hi = s_tab[2][2 * i + 1];
        x[0] = __vadd2(b3[0], lo.x); x[1] = __vadd2(b3[1], lo.y); x[2] = __vadd2(b3[2], lo.z); x[3] = __vadd2(b3[3], lo.w);
        x[4] = __vadd2(b3[4], hi.x); x[5] = __vadd2(b3[5], hi.y); x[6] = __vadd2(b3[6], hi.z); x[7] = __vadd2(b3[7], hi.w);
    }
    ch2_vgates(x, jv2);                                                     // b_2 over v^1
#pragma unroll
    for (int j = 0; j < 8; ++j) x[j] = __vadd2(x[j], T1[j]);               // a_1
    ch2_vgates(x, jv1);                                                     // b_1 over v^0
    // ---- level 0: G(u) = max_v ( B_0(u^0, v) + b_1[v] ) for the 8 elements of the lane's uint4
    unsigned g[8];
#pragma unroll
    for (int t = 0; t < 8; ++t) {
        unsigned acc = __vadd2(T0[t][0], x[0]);
#pragma unroll
        for (int j = 1; j < 8; ++j) acc = __viaddmax_s16x2(T0[t][j], x[j], acc);
        g[t] = __vmaxs2(acc, __byte_perm(acc, 0u, 0x1032));                 // both halves = G
    }
    uint4 G4;                                    // word k = elements t = 2k (lo), 2k + 1 (hi)
    G4.x = __byte_perm(g[0], g[1], 0x7610); G4.y = __byte_perm(g[2], g[3], 0x7610);
    G4.z = __byte_perm(g[4], g[5], 0x7610); G4.w = __byte_perm(g[6], g[7], 0x7610);
    return G4;
}

// b_3 of a tile: levels M-1 .. 3 (u^3 .. u^{M-1} = the bits of the tile index)
__device__ __forceinline__ void ch2_tile_b3(unsigned (&b3)[8], const unsigned long long tile, const int M,
                                            const uint4 (*s_tab)[32], const unsigned (*jv)[4]) {
#pragma unroll
    for (int j = 0; j < 8; ++j) b3[j] = 0u;
    for (int r = M - 1; r >= 3; --r) {
        const int ur = (int)((tile >> (4 * (r - 3))) & 15ull);
        const uint4 lo = s_tab[r][2 * ur], hi = s_tab[r][2 * ur + 1];
        b3[0] = __vadd2(b3[0], lo.x); b3[1] = __vadd2(b3[1], lo.y); b3[2] = __vadd2(b3[2], lo.z); b3[3] = __vadd2(b3[3], lo.w);
        b3[4] = __vadd2(b3[4], hi.x); b3[5] = __vadd2(b3[5], hi.y); b3[6] = __vadd2(b3[6], hi.z); b3[7] = __vadd2(b3[7], hi.w);
        const unsigned m2[4] = {jv[r][0], jv[r][1], jv[r][2], jv[r][3]};
        ch2_vgates(b3, m2);                                                 // -> b_r over v^{r-1}
    }
}

// A warp takes the tile pair (t, t + tiles / 2): the two tiles differ in the TOP bit of u, whose
// horizontal gate (ju_top, packed -2J; 0 in column 0) is applied here, before the column's diagonal --
// the gate-row passes in front of this kernel cover the bits below it.
__global__ void __launch_bounds__(CH2_WARPS * 32, 2) chimera_column_kernel(const ChimeraColumnParams q) {
    __shared__ uint4 s_tab[8][32];                    // [r][16 u x 2 uint4]
    __shared__ int s_max[CH2_WARPS];
    for (int i = threadIdx.x; i < q.M * 32; i += blockDim.x)
        s_tab[i >> 5][i & 31] = reinterpret_cast<const uint4*>(q.tables)[i];
    __syncthreads();
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    // the lane's rows of B_0 (u^0 = 8 (lane & 1) + t, t = 0..7) and its row of B_1 (u^1 = lane >> 1)
    unsigned T0[8][8], T1[8];
#pragma unroll
    for (int t = 0; t < 8; ++t) {
        const uint4 lo = s_tab[0][2 * (8 * (lane & 1) + t)], hi = s_tab[0][2 * (8 * (lane & 1) + t) + 1];
        T0[t][0] = lo.x; T0[t][1] = lo.y; T0[t][2] = lo.z; T0[t][3] = lo.w;
        T0[t][4] = hi.x; T0[t][5] = hi.y; T0[t][6] = hi.z; T0[t][7] = hi.w;
    }
    {
        const uint4 lo = s_tab[1][2 * (lane >> 1)], hi = s_tab[1][2 * (lane >> 1) + 1];
        T1[0] = lo.x; T1[1] = lo.y; T1[2] = lo.z; T1[3] = lo.w; T1[4] = hi.x; T1[5] = hi.y; T1[6] = hi.z; T1[7] = hi.w;
    }
    const unsigned jv1[4] = {q.jv[1][0], q.jv[1][1], q.jv[1][2], q.jv[1][3]};
    const unsigned jv2[4] = {q.jv[2][0], q.jv[2][1], q.jv[2][2], q.jv[2][3]};
    int best = -2147483647 - 1;
    const unsigned long long nw = (unsigned long long)gridDim.x * CH2_WARPS, half = q.tiles >> 1;
    for (unsigned long long tile = (unsigned long long)blockIdx.x * CH2_WARPS + warp; tile < half; tile += nw) {
        uint4* base0 = reinterpret_cast<uint4*>(q.state) + (tile << 9) + lane;      // 2^11 words = 2^9 uint4 per tile
        uint4* base1 = base0 + (half << 9);
        // the lane's 16 uint4 of either tile stream through two registers each
        uint4 n0 = make_uint4(0u, 0u, 0u, 0u), n1 = n0;
        if (!q.init) { n0 = base0[0]; n1 = base1[0]; }
        unsigned b30[8], b31[8];
        ch2_tile_b3(b30, tile, q.M, s_tab, q.jv);
        ch2_tile_b3(b31, tile + half, q.M, s_tab, q.jv);
#pragma unroll 1
        for (int i = 0; i < 16; ++i) {               // u^2 = i
            uint4 f0 = n0, f1 = n1;
            if (!q.init && i < 15) { n0 = base0[32 * (i + 1)]; n1 = base1[32 * (i + 1)]; }
            ch_gate(f0.x, f1.x, q.ju_top); ch_gate(f0.y, f1.y, q.ju_top);           // gate (A2) on the top bit of u
            ch_gate(f0.z, f1.z, q.ju_top); ch_gate(f0.w, f1.w, q.ju_top);
            const uint4 G0 = ch2_column_G(b30, i, s_tab, T0, T1, jv1, jv2);
            f0.x = __vadd2(f0.x, G0.x); f0.y = __vadd2(f0.y, G0.y); f0.z = __vadd2(f0.z, G0.z); f0.w = __vadd2(f0.w, G0.w);
            const uint4 G1 = ch2_column_G(b31, i, s_tab, T0, T1, jv1, jv2);
            f1.x = __vadd2(f1.x, G1.x); f1.y = __vadd2(f1.y, G1.y); f1.z = __vadd2(f1.z, G1.z); f1.w = __vadd2(f1.w, G1.w);
            if (q.reduce) {
                const unsigned m = __vmaxs2(__vmaxs2(__vmaxs2(f0.x, f0.y), __vmaxs2(f0.z, f0.w)),
                                            __vmaxs2(__vmaxs2(f1.x, f1.y), __vmaxs2(f1.z, f1.w)));
                const int lo = (int)(short)(m & 0xffffu), hi = (int)(short)(m >> 16);
                best = max(best, max(lo, hi));
            } else {
                base0[32 * i] = f0; base1[32 * i] = f1;
            }
        }
    }
    if (q.reduce) {
        for (int o = 16; o; o >>= 1) best = max(best, __shfl_xor_sync(0xffffffffu, best, o));
        if (lane == 0) s_max[warp] = best;
        __syncthreads();
        if (threadIdx.x == 0) {
            for (int w = 1; w < CH2_WARPS; ++w) best = max(best, s_max[w]);
            atomicMax(q.out, best);
        }
    }
}

}  // namespace ttn

// =============================================================================================
// CountingTropical form (Eq. (4); the chimera entropies of PAPER.md:128, Fig. 3): the
// same column sweep with elements (x f32, n f64), structure of arrays.  The horizontal couplings run
// as one gate row on the counting Ising pass kernels (ttn_fcount.cuh); the column's vertical chain
// is contracted on the fly in CountingTropical arithmetic:
//     (x, n) (+) (y, m) = (max, counts added on exact ties),   (x, n) (.) (y, m) = (x + y, n m),
//     F[u] <- F[u] (.) G_c(u),   G_c(u) = (+)_{v^0..v^{M-1}} (.)_r B_r(u^r, v^r) (.) V_{r-1}(v^{r-1}, v^r).
// Couplings are integers (the caller checks), so f32 sums are exact and ties are exact ties.
// Same tile as the Tropical<i16> kernel: a warp owns (u^0, u^1, u^2), lane = (bit 3 of u^0, u^1), the lane's
// elements of one u^2 value are 8 consecutive floats / doubles.
namespace ttn {

struct ChimeraCountParams {
    float* x; double* n;          // 2^(4M) elements each
    int M;                        // rows of cells, 3 <= M <= 8
    int init, reduce;
    unsigned long long tiles;     // 2^(4M-12)
    const float* tables;          // [M rows][16 u][16 v]: B_r(u, v) of this column
    float jv[8][4];               // [r][k] = -2 Jv[r-1][c][k]; row 0 unused
    float* part_x; double* part_n;   // [gridDim.x] (reduce)
    double n_scale;               // a power of two put on every count of this column (1.0, or 2^-8p for p padded rows)
};

__device__ __forceinline__ double ch2_ind(bool p) { return __hiloint2double(p ? 0x3ff00000 : 0, 0); }

// the four single-spin counting gates of one vertical coupling group on a 16-vector over v
__device__ __forceinline__ void ch2_cvgates(float (&x)[16], double (&n)[16], const float* m2) {
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const int B = 1 << k;
        const float m = m2[k];
#pragma unroll
        for (int v = 0; v < 16; ++v) {
            if (v & B) continue;
            const float xa = x[v], xb = x[v | B];
            const double na = n[v], nb = n[v | B];
            const float ca = xb + m, cb = xa + m;
            n[v] = fma(nb, ch2_ind(ca >= xa), na * ch2_ind(xa >= ca));
            n[v | B] = fma(na, ch2_ind(cb >= xb), nb * ch2_ind(xb >= cb));
            x[v] = fmaxf(xa, ca);
            x[v | B] = fmaxf(xb, cb);
        }
    }
}

constexpr int CH2C_WARPS = 8;

__global__ void __launch_bounds__(CH2C_WARPS * 32, 1) chimera_column_count_kernel(const ChimeraCountParams q) {
    __shared__ float s_tab[8][16][16];
    __shared__ float s_jv[8][4];
    __shared__ float s_redx[CH2C_WARPS];
    __shared__ double s_redn[CH2C_WARPS];
    for (int i = threadIdx.x; i < q.M * 256; i += blockDim.x) (&s_tab[0][0][0])[i] = q.tables[i];
    if (threadIdx.x < 32) (&s_jv[0][0])[threadIdx.x] = q.jv[threadIdx.x >> 2][threadIdx.x & 3];
    __syncthreads();
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int u1 = lane >> 1, u0hi = 8 * (lane & 1);
    float best = -INFINITY; double bcnt = 0.0;
    const unsigned long long nw = (unsigned long long)gridDim.x * CH2C_WARPS;
    for (unsigned long long tile = (unsigned long long)blockIdx.x * CH2C_WARPS + warp; tile < q.tiles; tile += nw) {
        // ---- levels M-1 .. 3: uniform per tile
        float b3x[16]; double b3n[16];
#pragma unroll
        for (int v = 0; v < 16; ++v) { b3x[v] = 0.f; b3n[v] = q.n_scale; }     // every count below is linear in it
        for (int r = q.M - 1; r >= 3; --r) {
            const int ur = (int)((tile >> (4 * (r - 3))) & 15ull);
#pragma unroll
            for (int v = 0; v < 16; ++v) b3x[v] += s_tab[r][ur][v];
            ch2_cvgates(b3x, b3n, s_jv[r]);
        }
        float* px = q.x + (tile << 12) + 8 * lane;
        double* pn = q.n + (tile << 12) + 8 * lane;
#pragma unroll 1
        for (int i = 0; i < 16; ++i) {               // u^2 = i
            float fx[8]; double fn[8];
            if (!q.init) {
                const float4 a = *reinterpret_cast<const float4*>(px + 256 * i), b = *reinterpret_cast<const float4*>(px + 256 * i + 4);
                fx[0] = a.x; fx[1] = a.y; fx[2] = a.z; fx[3] = a.w; fx[4] = b.x; fx[5] = b.y; fx[6] = b.z; fx[7] = b.w;
#pragma unroll
                for (int t = 0; t < 8; t += 2) {
                    const double2 d = *reinterpret_cast<const double2*>(pn + 256 * i + t);
                    fn[t] = d.x; fn[t + 1] = d.y;
                }
            } else {
#pragma unroll
                for (int t = 0; t < 8; ++t) { fx[t] = 0.f; fn[t] = 1.0; }
            }
            float x[16]; double n[16];
#pragma unroll
            for (int v = 0; v < 16; ++v) { x[v] = b3x[v] + s_tab[2][i][v]; n[v] = b3n[v]; }
            ch2_cvgates(x, n, s_jv[2]);                                             // b_2 over v^1
#pragma unroll
            for (int v = 0; v < 16; ++v) x[v] += s_tab[1][u1][v];                   // a_1
            ch2_cvgates(x, n, s_jv[1]);                                             // b_1 over v^0
#pragma unroll
            for (int t = 0; t < 8; ++t) {            // G(u) = (+)_v B_0(u^0, v) (.) b_1[v]
                float c[16];
                float g = -INFINITY;
#pragma unroll
                for (int v = 0; v < 16; ++v) { c[v] = s_tab[0][u0hi + t][v] + x[v]; g = fmaxf(g, c[v]); }
                double gn = 0.0;
#pragma unroll
                for (int v = 0; v < 16; ++v) gn = fma(n[v], ch2_ind(c[v] == g), gn);
                fx[t] += g; fn[t] *= gn;
            }
            if (q.reduce) {
#pragma unroll
                for (int t = 0; t < 8; ++t) {
                    if (fx[t] > best) { best = fx[t]; bcnt = fn[t]; } else if (fx[t] == best) bcnt += fn[t];
                }
            } else {
                *reinterpret_cast<float4*>(px + 256 * i) = make_float4(fx[0], fx[1], fx[2], fx[3]);
                *reinterpret_cast<float4*>(px + 256 * i + 4) = make_float4(fx[4], fx[5], fx[6], fx[7]);
#pragma unroll
                for (int t = 0; t < 8; t += 2) *reinterpret_cast<double2*>(pn + 256 * i + t) = make_double2(fn[t], fn[t + 1]);
            }
        }
    }
    if (q.reduce) {
        float m = best;
        for (int o = 16; o; o >>= 1) m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, o));
        double c = best == m ? bcnt : 0.0;
        for (int o = 16; o; o >>= 1) c += __shfl_xor_sync(0xffffffffu, c, o);
        if (lane == 0) { s_redx[warp] = m; s_redn[warp] = c; }
        __syncthreads();
        if (threadIdx.x == 0) {
            float mm = s_redx[0];
            for (int w = 1; w < CH2C_WARPS; ++w) mm = fmaxf(mm, s_redx[w]);
            double cc = 0.0;
            for (int w = 0; w < CH2C_WARPS; ++w) if (s_redx[w] == mm) cc += s_redn[w];
            q.part_x[blockIdx.x] = mm; q.part_n[blockIdx.x] = cc;
        }
    }
}

}  // namespace ttn
