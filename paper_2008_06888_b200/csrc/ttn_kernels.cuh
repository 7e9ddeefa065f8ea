// ttn_kernels.cuh -- device side of the tropical transfer sweep, generic tile path: every
// semiring (Tropical<f32>, CountingTropical<f32,f64>), q = 2 (Ising) and q = 3 (Potts), and
// the checkpointed ground-configuration call.
//
// One launch of pass_kernel = one HBM pass over the q^L state: each
// CTA stages one tile (digits [0,lo) U [a,b) of the state index) in shared memory, applies the
// pass's gate list as butterflies over the gate's digit, and writes the tile back in place
// ("all operations should be performed inplace").  The first pass is write-only
// (initial state (0,0)^{(x)L}), the last is read-only and fuses the final
// (+)-reduction.
//
// DIAGONAL FRAME (planner.h): the sweep runs on V'' with V = A_r V'', A_r the accumulated row
// diagonals (A3), (A4) PAPER.md:247-252, so no diagonal is ever applied to the state; each gate
// (A2) PAPER.md:242 / the 3x3 Potts gate of App. C PAPER.md:296 is conjugated with A_{r-1}:
//   Ising:  a' = a (+) (b (.) ka[nl][nr]),  b' = b (+) (a (.) kb[nl][nr])          (8 constants)
//   Potts:  y[t] = x[t] (.) R(t),  new[t'] = ( (+)_t y[t] (.) Jv delta(t,t') ) (.) (-R(t')),
//           R(t) = Kl delta(t_{c-1}, t) + Kr delta(t, t_{c+1})                      (3 constants)
// with nl, nr / t_{c-1}, t_{c+1} the neighbour digits of the element's own index.  The last
// pass multiplies by A_{L-1}(s) before the reduction; the configuration call keeps V'' in its
// checkpoints and the backward pass adds A_r(s).
//
// Semirings: Tropical<f32>: x (+) y = max, x (.) y = x + y (Eq. (2)
// PAPER.md:57); CountingTropical<f32,f64>: Eq. (4), counts summed on exact ties.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>
#include "planner.h"

namespace ttn {

constexpr int GMAX_L = 64;          // digits (columns) supported by the generic kernels' tables

struct PassParams {
    int L, T, lo, a, b;
    unsigned long long P_lo, P_a, P_mid, P_b;   // q^lo, q^a, q^(a-lo), q^b
    unsigned int n_tile;                          // q^T elements per tile
    unsigned long long tiles_per_inst;            // q^(L-T)
    const float* src_x; float* dst_x;             // instance 0 base pointers
    const double* src_n; double* dst_n;           // counting only
    unsigned long long src_stride, dst_stride;    // elements between instances
    const Op* ops; int n_ops;                     // this pass's gates
    const float* gate_k;                          // [inst][all gates][8]; this pass's slice of instance 0
    unsigned long long gate_inst_stride;          // floats between instances
    const float* fin;                             // [inst][2 * GMAX_L]: H_c, K_c of A_{L-1} (REDUCE pass)
    int flags;
    float* part_x; double* part_n;                // [inst][tile] partial reductions
    int z3;                                       // q = 3, colour-rotation reduction (planner.h): L, T and every power
                                                  // above count the STORED digits (digit d = column d + 1); a CTA holds
                                                  // the three tiles of a rotation orbit; ops with pos = VCOL act on column 0
};

// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ float warp_max(float v) {
    for (int o = 16; o; o >>= 1) v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
}
__device__ __forceinline__ double warp_sum(double v) {
    for (int o = 16; o; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// tropical / counting (+) of candidate (cx, cn) into accumulator (x, n): Eq. (4)
template <bool COUNT>
__device__ __forceinline__ void oplus(float& x, double& n, float cx, double cn) {
    if (COUNT) {          // branch-free: the sum is formed always and selected on the exact tie
        const double s = n + cn;
        n = cx > x ? cn : (cx == x ? s : n);
    }
    x = fmaxf(x, cx);
}

// 3-input max: one FMNMX3 on sm_100
__device__ __forceinline__ float max3(float a, float b, float c) {
    float r; asm("max.f32 %0, %1, %2, %3;" : "=f"(r) : "f"(a), "f"(b), "f"(c)); return r;
}
// 1.0 / 0.0 from a predicate (only the high word of the double is selected)
__device__ __forceinline__ double ind01(bool p) { return __hiloint2double(p ? 0x3ff00000 : 0, 0); }

// exact n / d for n * d < 2^32 with the host-side magic M = floor(2^32 / d) + 1
__device__ __forceinline__ unsigned fastdiv(unsigned n, unsigned magic) { return __umulhi(n, magic); }
__host__ __device__ inline unsigned fastdiv_magic(unsigned d) { return d <= 1 ? 0u : (unsigned)(0x100000000ull / d) + 1u; }

// column held by tile position p
__device__ __forceinline__ int tile_col(const PassParams& p, int pos) { return pos < p.lo ? pos : p.a + (pos - p.lo); }

// weight of the accumulated diagonal A(s) = sum_c H_c f1(d_c) + sum_c K_c f2(d_c, d_{c+1})
template <int Q> __device__ __forceinline__ float diag1(float H, int d) { return Q == 2 ? (d ? -H : H) : 0.f; }
template <int Q> __device__ __forceinline__ float diag2(float K, int d0, int d1) {
    return Q == 2 ? (d0 == d1 ? K : -K) : (d0 == d1 ? K : 0.f);
}

template <int Q, bool COUNT>
__global__ void __launch_bounds__(512) pass_kernel(const PassParams p) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double* sn = reinterpret_cast<double*>(smem_raw);                       // [n_tile] if COUNT
    float* sx = reinterpret_cast<float*>(smem_raw + (COUNT ? (size_t)p.n_tile * 8 : 0));
    __shared__ int s_dig[GMAX_L];            // digits of this tile's base index (columns outside the tile)
    __shared__ float s_fin[2 * GMAX_L];      // H_c, K_c of A_{L-1} (REDUCE pass)
    __shared__ float s_aout;                 // part of A_{L-1} that only involves columns outside the tile
    const unsigned N = p.n_tile;
    const unsigned long long gtile = blockIdx.x;
    const unsigned long long inst = gtile / p.tiles_per_inst;
    const unsigned long long tile = gtile % p.tiles_per_inst;
    const unsigned long long base = (tile % p.P_mid) * p.P_lo + (tile / p.P_mid) * p.P_b;
    const unsigned plo = (unsigned)p.P_lo;

    // ---- load (or initialise to the semiring one) -------------------------------------------
    if (p.flags & PASS_INIT) {
        for (unsigned t = threadIdx.x; t < N; t += blockDim.x) { sx[t] = 0.f; if (COUNT) sn[t] = 1.0; }
    } else {
        const float* gx = p.src_x + inst * p.src_stride + base;
        const double* gn = COUNT ? p.src_n + inst * p.src_stride + base : nullptr;
        for (unsigned t = threadIdx.x; t < N; t += blockDim.x) {
            unsigned long long off = (unsigned long long)(t % plo) + (unsigned long long)(t / plo) * p.P_a;
            sx[t] = gx[off];
            if (COUNT) sn[t] = gn[off];
        }
    }
    for (int i = threadIdx.x; i < p.L; i += blockDim.x) {   // digit c of the base index (0 for the tile's own columns)
        unsigned long long s = base;
        for (int c = 0; c < i; ++c) s /= Q;
        s_dig[i] = (int)(s % Q);
    }
    if (p.flags & PASS_REDUCE)
        for (int i = threadIdx.x; i < 2 * GMAX_L; i += blockDim.x) s_fin[i] = p.fin[inst * (2 * GMAX_L) + i];
    __syncthreads();

    // ---- gate list -------------------------------------------------------------------------------
    // Per-gate index constants (digit weight, division magics, where the neighbour digits come
    // from) are computed once per gate by ONE thread each into shared memory, not by every thread
    // (the 64-bit division behind fastdiv_magic is a subroutine call).
    constexpr int GCHUNK = 256;
    __shared__ uint4 s_aux[GCHUNK];          // x = st, y = magic(st), z = magic(st / Q), w = flags
    const float* GK = p.gate_k + inst * p.gate_inst_stride;
    for (int k = 0; k < p.n_ops; ++k) {
        if (k % GCHUNK == 0) {
            for (int i = threadIdx.x; i < GCHUNK && k + i < p.n_ops; i += blockDim.x) {
                const Op o = p.ops[k + i];
                unsigned s_ = 1;
                for (int j = 0; j < o.pos; ++j) s_ *= Q;
                const unsigned sq = o.pos > 0 ? s_ / Q : 1;
                const bool li = o.pos > 0 && tile_col(p, o.pos - 1) == o.c - 1;
                const bool ri = o.pos + 1 < p.T && tile_col(p, o.pos + 1) == o.c + 1;
                const int dlo = o.c > 0 ? s_dig[o.c - 1] : 0, dro = o.c + 1 < p.L ? s_dig[o.c + 1] : 0;
                s_aux[i] = make_uint4(s_, fastdiv_magic(s_), fastdiv_magic(sq),
                                      (unsigned)li | ((unsigned)ri << 1) | ((unsigned)dlo << 2) | ((unsigned)dro << 4));
            }
            __syncthreads();
        }
        const Op op = p.ops[k];
        const int pos = op.pos;
        const uint4 aux = s_aux[k % GCHUNK];
        const unsigned st = aux.x, m_st = aux.y, m_stq = aux.z;
        const unsigned st_q = pos > 0 ? st / Q : 1;
        const bool l_in = aux.w & 1u, r_in = (aux.w >> 1) & 1u;
        const int dl_out = (int)((aux.w >> 2) & 3u), dr_out = (int)((aux.w >> 4) & 3u);
        const float4 k0 = reinterpret_cast<const float4*>(GK)[2 * k], k1 = reinterpret_cast<const float4*>(GK)[2 * k + 1];
        const unsigned ngrp = N / Q;
        for (unsigned g = threadIdx.x; g < ngrp; g += blockDim.x) {
            unsigned hi, lo; int dl, dr;
            if (Q == 2) {
                hi = g >> pos; lo = g & (st - 1);
                dl = l_in ? (int)(lo >> (pos - 1)) : dl_out;                               // top digit of lo
                dr = r_in ? (int)(hi & 1u) : dr_out;
            } else {
                hi = st == 1 ? g : fastdiv(g, m_st); lo = g - hi * st;
                dl = l_in ? (int)(st_q == 1 ? lo : fastdiv(lo, m_stq)) : dl_out;
                dr = r_in ? (int)(hi % Q) : dr_out;
            }
            const unsigned i0 = hi * (st * Q) + lo;
            if (Q == 2) {
                // conjugated (A2): a' = a (+) (b + ka[dl][dr]),  b' = b (+) (a + kb[dl][dr])
                const int n = dl * 2 + dr;
                const float ka = n == 0 ? k0.x : (n == 1 ? k0.y : (n == 2 ? k0.z : k0.w));
                const float kb = n == 0 ? k1.x : (n == 1 ? k1.y : (n == 2 ? k1.z : k1.w));
                float xa = sx[i0], xb = sx[i0 + st];
                const float ca = xb + ka, cb = xa + kb;
                if (COUNT) {
                    const double na = sn[i0], nb = sn[i0 + st];
                    float ya = xa; double ma = na; oplus<true>(ya, ma, ca, nb);
                    float yb = xb; double mb = nb; oplus<true>(yb, mb, cb, na);
                    sx[i0] = ya; sx[i0 + st] = yb; sn[i0] = ma; sn[i0 + st] = mb;
                } else {
                    sx[i0] = fmaxf(xa, ca); sx[i0 + st] = fmaxf(xb, cb);
                }
            } else {
                // conjugated Potts gate: k0 = (Jv, Kl, Kr, -)
                const float J = k0.x, Kl = k0.y, Kr = k0.z;
                float R[3], x[3];
#pragma unroll
                for (int t = 0; t < 3; ++t) {
                    R[t] = (t == dl ? Kl : 0.f) + (t == dr ? Kr : 0.f);
                    x[t] = sx[i0 + t * st] + R[t];
                }
                if (COUNT) {
                    // Eq. (4) over three candidates: count = sum of n_t over the exact maximisers; the
                    // 0/1 indicators make it FP64 multiply-adds instead of 64-bit selects
                    double n[3];
#pragma unroll
                    for (int t = 0; t < 3; ++t) n[t] = sn[i0 + t * st];
#pragma unroll
                    for (int tn = 0; tn < 3; ++tn) {
                        float c[3];
#pragma unroll
                        for (int t = 0; t < 3; ++t) c[t] = t == tn ? x[t] + J : x[t];
                        const float best = max3(c[0], c[1], c[2]);
                        const double m = fma(n[2], ind01(c[2] == best), fma(n[1], ind01(c[1] == best), n[0] * ind01(c[0] == best)));
                        sx[i0 + tn * st] = best - R[tn]; sn[i0 + tn * st] = m;
                    }
                } else {
                    sx[i0] = max3(x[0] + J, x[1], x[2]) - R[0];
                    sx[i0 + st] = max3(x[1] + J, x[0], x[2]) - R[1];
                    sx[i0 + 2 * st] = max3(x[2] + J, x[0], x[1]) - R[2];
                }
            }
        }
        __syncthreads();
    }

    // ---- store, or multiply by A_{L-1}(s) and reduce ----------------------------------------------
    if (p.flags & PASS_REDUCE) {
        const float* H = s_fin; const float* K = s_fin + GMAX_L;
        if (threadIdx.x == 0) {              // terms whose columns all lie outside the tile
            float acc = 0.f;
            for (int c = 0; c < p.L; ++c) {
                const bool in_c = c < p.lo || (c >= p.a && c < p.b);
                if (!in_c) acc += diag1<Q>(H[c], s_dig[c]);
                if (c + 1 < p.L) {
                    const bool in_n = c + 1 < p.lo || (c + 1 >= p.a && c + 1 < p.b);
                    if (!in_c && !in_n) acc += diag2<Q>(K[c], s_dig[c], s_dig[c + 1]);
                }
            }
            s_aout = acc;
        }
        __syncthreads();
        float mx = -INFINITY;
        for (unsigned t = threadIdx.x; t < N; t += blockDim.x) {
            // walk the tile-local digits of t: position pos holds column tile_col(pos)
            float acc = s_aout;
            unsigned rest = t;
            int dprev = 0, cprev = -2;
            for (int pos = 0; pos < p.T; ++pos) {
                const int d = (int)(rest % Q); rest /= Q;
                const int c = tile_col(p, pos);
                acc += diag1<Q>(H[c], d);
                if (c > 0) {
                    if (cprev == c - 1) acc += diag2<Q>(K[c - 1], dprev, d);           // left neighbour in the tile
                    else acc += diag2<Q>(K[c - 1], s_dig[c - 1], d);                   // left neighbour outside
                }
                const bool right_in = pos + 1 < p.T && tile_col(p, pos + 1) == c + 1;
                if (c + 1 < p.L && !right_in) acc += diag2<Q>(K[c], d, s_dig[c + 1]);  // right neighbour outside
                dprev = d; cprev = c;
            }
            const float val = sx[t] + acc;
            sx[t] = val;
            mx = fmaxf(mx, val);
        }
        __shared__ float red_x[16];
        __shared__ double red_n[16];
        mx = warp_max(mx);
        if ((threadIdx.x & 31) == 0) red_x[threadIdx.x >> 5] = mx;
        __syncthreads();
        float bm = red_x[0];
        for (int w = 1; w < (int)(blockDim.x >> 5); ++w) bm = fmaxf(bm, red_x[w]);
        double cnt = 0.0;
        if (COUNT) {
            for (unsigned t = threadIdx.x; t < N; t += blockDim.x) if (sx[t] == bm) cnt += sn[t];
            cnt = warp_sum(cnt);
            if ((threadIdx.x & 31) == 0) red_n[threadIdx.x >> 5] = cnt;
            __syncthreads();
        }
        if (threadIdx.x == 0) {
            p.part_x[gtile] = bm;
            if (COUNT) {
                double tot = 0.0;
                for (int w = 0; w < (int)(blockDim.x >> 5); ++w) tot += red_n[w];
                p.part_n[gtile] = tot;
            }
        }
    } else {
        float* gx = p.dst_x + inst * p.dst_stride + base;
        double* gn = COUNT ? p.dst_n + inst * p.dst_stride + base : nullptr;
        for (unsigned t = threadIdx.x; t < N; t += blockDim.x) {
            unsigned long long off = (unsigned long long)(t % plo) + (unsigned long long)(t / plo) * p.P_a;
            gx[off] = sx[t];
            if (COUNT) gn[off] = sn[t];
        }
    }
}

// Final (+) over the per-tile partials of each instance; fixed order => deterministic f64 sum.
template <bool COUNT>
__global__ void __launch_bounds__(256) final_reduce_kernel(const float* part_x, const double* part_n,
                                                           unsigned long long tiles_per_inst,
                                                           float* out_x, double* out_n) {
    const unsigned long long inst = blockIdx.x;
    const float* px = part_x + inst * tiles_per_inst;
    float mx = -INFINITY;
    for (unsigned long long i = threadIdx.x; i < tiles_per_inst; i += blockDim.x) mx = fmaxf(mx, px[i]);
    __shared__ float red_x[8];
    __shared__ double red_n[8];
    mx = warp_max(mx);
    if ((threadIdx.x & 31) == 0) red_x[threadIdx.x >> 5] = mx;
    __syncthreads();
    float bm = red_x[0];
    for (int w = 1; w < 8; ++w) bm = fmaxf(bm, red_x[w]);
    double cnt = 0.0;
    if (COUNT) {
        const double* pn = part_n + inst * tiles_per_inst;
        for (unsigned long long i = threadIdx.x; i < tiles_per_inst; i += blockDim.x) if (px[i] == bm) cnt += pn[i];
        cnt = warp_sum(cnt);
        if ((threadIdx.x & 31) == 0) red_n[threadIdx.x >> 5] = cnt;
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        out_x[inst] = bm;
        if (COUNT) { double tot = 0.0; for (int w = 0; w < 8; ++w) tot += red_n[w]; out_n[inst] = tot; }
    }
}

// ---------------------------------------------------------------------------------------------
// Backtrace ("caching intermediate contraction results and
// backtracking").  The checkpoints hold V''_r (diagonal frame), V_r = A_r V''_r, so
//   s_{L-1} = argmax_s ( C_{L-1}[s] + A_{L-1}(s) ),
//   s_r     = argmax_s ( C_r[s] + A_r(s) + sum_c Jv[r][c] sigma_c(s) sigma_c(s_{r+1}) ).
// Lowest index wins ties (footnote [49] PAPER.md:201).
struct ArgmaxParams {
    int L, r, has_next, nblk;
    unsigned long long NS;
    const float* C;                     // checkpoint C_r of instance 0
    unsigned long long c_stride;        // elements between instances
    const float* Jh; const float* Jv; const float* h;   // device couplings (per instance); h may be null
    const unsigned long long* s_next;   // [batch] state of row r+1 (if has_next)
    float* part_v; unsigned long long* part_s;   // [batch][nblk]
    unsigned long long* s_out;          // [batch]
    float* v_out;                       // [batch] max value (written when !has_next)
    signed char* sigma;                 // [batch][L][L]
};

__device__ __forceinline__ void argmax_combine(float& v, unsigned long long& s, float v2, unsigned long long s2) {
    if (v2 > v || (v2 == v && s2 < s)) { v = v2; s = s2; }
}

// Z2 (h = 0, checkpoints are half-states over u = (s_1 .. s_{L-1}), column 0 up): the candidates of a row
// are s = (0, u) with value C[u] + A(u) + Wj(u) and its flip (1, ~u), whose checkpoint entry is the same
// (W[1, ~u] = W[0, u]), whose A is the same (no field) and whose bond term to the next row is -Wj(u):
//     best of the pair = C[u] + A(u) + |Wj(u)|,   s = (0, u) if Wj(u) >= 0 else its global flip.
template <bool Z2>
__global__ void __launch_bounds__(256) argmax_partial_kernel(const ArgmaxParams p) {
    const unsigned long long inst = blockIdx.y;
    __shared__ float jsig[GMAX_L];      // coefficient of sigma_c: Jv sigma'_c + H_c (accumulated through row r)
    __shared__ float kacc[GMAX_L];      // coefficient of sigma_c sigma_{c+1}
    if (threadIdx.x < p.L) {
        const int c = threadIdx.x, L = p.L;
        double hs = 0.0, ks = 0.0;
        for (int rr = 0; rr <= p.r; ++rr) {
            if (p.h) hs += (double)p.h[inst * (unsigned long long)(L * L) + rr * L + c];
            if (c + 1 < L) ks += (double)p.Jh[inst * (unsigned long long)(L * (L - 1)) + rr * (L - 1) + c];
        }
        double j = 0.0;
        if (p.has_next) {
            j = (double)p.Jv[inst * (unsigned long long)((L - 1) * L) + p.r * L + c];
            if ((p.s_next[inst] >> c) & 1ull) j = -j;
        }
        jsig[c] = (float)(j + hs);
        kacc[c] = (float)ks;
    }
    __syncthreads();
    // w(s) = sum_c jsig[c] sigma_c + sum_c kacc[c] sigma_c sigma_{c+1}, split into one 256-entry
    // table per byte of s (terms inside the byte) + one sign per byte boundary
    __shared__ float tab[4][256];                    // L <= 32 (four bytes of s)
    __shared__ float tabj[Z2 ? 4 : 1][256];          // Z2: the bond-to-next-row part on its own (tab holds A only)
    const int nchunk = (p.L + 7) >> 3;
    for (int m = 0; m < nchunk; ++m) {
        const int v = threadIdx.x;                   // blockDim.x = 256
        float acc = 0.f, accj = 0.f;
        for (int i = 0; i < 8 && 8 * m + i < p.L; ++i) {
            const int c = 8 * m + i, b = (v >> i) & 1;
            if (Z2) accj += b ? -jsig[c] : jsig[c]; else acc += b ? -jsig[c] : jsig[c];
            if (i + 1 < 8 && c + 1 < p.L) acc += (b == ((v >> (i + 1)) & 1)) ? kacc[c] : -kacc[c];
        }
        tab[m][v] = acc;
        if (Z2) tabj[m][v] = accj;
    }
    __syncthreads();
    const float* C = p.C + inst * p.c_stride;
    float bv = -INFINITY; unsigned long long bs = ~0ull;
    const unsigned long long full = (p.L >= 64) ? ~0ull : ((1ull << p.L) - 1ull);
    for (unsigned long long e = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; e < p.NS;
         e += (unsigned long long)gridDim.x * blockDim.x) {
        const unsigned long long s = Z2 ? e << 1 : e;         // Z2: e = u, the full index has column 0 up
        const unsigned long long x = s ^ (s >> 1);            // bit c set <=> sigma_c != sigma_{c+1}
        float w = tab[0][s & 255u], wj = Z2 ? tabj[0][s & 255u] : 0.f;
        for (int m = 1; m < nchunk; ++m) {
            w += tab[m][(s >> (8 * m)) & 255u];
            if (Z2) wj += tabj[m][(s >> (8 * m)) & 255u];
            w += ((x >> (8 * m - 1)) & 1ull) ? -kacc[8 * m - 1] : kacc[8 * m - 1];
        }
        if (Z2) argmax_combine(bv, bs, C[e] + (w + fabsf(wj)), wj >= 0.f ? s : (~s & full));
        else argmax_combine(bv, bs, C[s] + w, s);
    }
    for (int o = 16; o; o >>= 1) {
        float v2 = __shfl_xor_sync(0xffffffffu, bv, o);
        unsigned long long s2 = __shfl_xor_sync(0xffffffffu, bs, o);
        argmax_combine(bv, bs, v2, s2);
    }
    __shared__ float rv[8];
    __shared__ unsigned long long rs[8];
    if ((threadIdx.x & 31) == 0) { rv[threadIdx.x >> 5] = bv; rs[threadIdx.x >> 5] = bs; }
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int w = 1; w < 8; ++w) argmax_combine(bv, bs, rv[w], rs[w]);
        p.part_v[inst * p.nblk + blockIdx.x] = bv;
        p.part_s[inst * p.nblk + blockIdx.x] = bs;
    }
}

__global__ void __launch_bounds__(32) argmax_final_kernel(const ArgmaxParams p) {
    const unsigned long long inst = blockIdx.x;
    float bv = -INFINITY; unsigned long long bs = ~0ull;
    for (int i = threadIdx.x; i < p.nblk; i += 32) argmax_combine(bv, bs, p.part_v[inst * p.nblk + i], p.part_s[inst * p.nblk + i]);
    for (int o = 16; o; o >>= 1) {
        float v2 = __shfl_xor_sync(0xffffffffu, bv, o);
        unsigned long long s2 = __shfl_xor_sync(0xffffffffu, bs, o);
        argmax_combine(bv, bs, v2, s2);
    }
    if (threadIdx.x == 0) { p.s_out[inst] = bs; if (!p.has_next) p.v_out[inst] = bv; }
    if (threadIdx.x < p.L)
        p.sigma[(inst * p.L + p.r) * p.L + threadIdx.x] = ((bs >> threadIdx.x) & 1ull) ? -1 : 1;
}

// Whole backtrace of one instance in ONE CTA (small lattices in batches, cfg 2): rows L-1 .. 0 are
// inherently sequential (s_r needs s_{r+1}) but instances are independent, so a CTA walks the L
// checkpoints of its instance without any launch or grid synchronisation in between.  Same
// arithmetic, in the same order, as argmax_partial_kernel + argmax_final_kernel (the prefix sums
// H_c, K_c over rows are formed once, in f64, in the same row order).
constexpr int BT_THREADS = 512;
constexpr int BT_MAX_L = 20;            // 2^20 states per row per CTA at most

__global__ void __launch_bounds__(BT_THREADS) backtrace_inst_kernel(const ArgmaxParams p) {
    const unsigned long long inst = blockIdx.x;
    const int L = p.L;
    __shared__ double hsum[BT_MAX_L][BT_MAX_L];   // [r][c] = sum_{rr <= r} h[rr][c]
    __shared__ double ksum[BT_MAX_L][BT_MAX_L];   // [r][c] = sum_{rr <= r} Jh[rr][c]
    __shared__ float jsig[BT_MAX_L], kacc[BT_MAX_L];
    __shared__ __align__(16) float tab[3][256];
    __shared__ float rv[BT_THREADS / 32];
    __shared__ unsigned long long rs[BT_THREADS / 32];
    __shared__ unsigned long long s_next;
    if (threadIdx.x < L) {
        const int c = threadIdx.x;
        double hs = 0.0, ks = 0.0;
        for (int rr = 0; rr < L; ++rr) {
            if (p.h) hs += (double)p.h[inst * (unsigned long long)(L * L) + rr * L + c];
            if (c + 1 < L) ks += (double)p.Jh[inst * (unsigned long long)(L * (L - 1)) + rr * (L - 1) + c];
            hsum[rr][c] = hs; ksum[rr][c] = ks;
        }
    }
    __syncthreads();
    const int nchunk = (L + 7) >> 3;
    for (int r = L - 1; r >= 0; --r) {
        const bool has_next = r < L - 1;
        if (threadIdx.x < L) {
            const int c = threadIdx.x;
            double j = 0.0;
            if (has_next) {
                j = (double)p.Jv[inst * (unsigned long long)((L - 1) * L) + r * L + c];
                if ((s_next >> c) & 1ull) j = -j;
            }
            jsig[c] = (float)(j + hsum[r][c]);
            kacc[c] = (float)ksum[r][c];
        }
        __syncthreads();
        for (int e = threadIdx.x; e < nchunk * 256; e += BT_THREADS) {
            const int m = e >> 8, v = e & 255;
            float acc = 0.f;
            for (int i = 0; i < 8 && 8 * m + i < L; ++i) {
                const int c = 8 * m + i, b = (v >> i) & 1;
                acc += b ? -jsig[c] : jsig[c];
                if (i + 1 < 8 && c + 1 < L) acc += (b == ((v >> (i + 1)) & 1)) ? kacc[c] : -kacc[c];
            }
            tab[m][v] = acc;
        }
        __syncthreads();
        const float* C = p.C + inst * p.c_stride + (unsigned long long)r * p.NS;
        float bv = -INFINITY; unsigned long long bs = ~0ull;
        // w(s) term by term in the order of argmax_partial_kernel: tab[0], then per higher byte
        // its table entry and the boundary bond.  A thread visits its states in increasing order,
        // so "lowest index wins ties" is a strict > inside the thread (NS <= 2^20: 32-bit indices).
        const unsigned ns = (unsigned)p.NS;
        unsigned b32 = 0xffffffffu;
        auto visit = [&](float c, unsigned s) {
            const unsigned x = s ^ (s >> 1);                      // bit c set <=> sigma_c != sigma_{c+1}
            float w = tab[0][s & 255u];
            for (int m = 1; m < nchunk; ++m) {
                w += tab[m][(s >> (8 * m)) & 255u];
                w += ((x >> (8 * m - 1)) & 1u) ? -kacc[8 * m - 1] : kacc[8 * m - 1];
            }
            const float v = c + w;
            if (v > bv) { bv = v; b32 = s; }
        };
        if (ns >= 4u * BT_THREADS) {              // 16-byte loads, four in flight per thread
            // The four states of a float4 differ in bits 0, 1 only: the table entries of the higher bytes and
            // the boundary bonds are fetched once per float4, tab[0] with one 128-bit load; every element's
            // sum is formed in the order of visit() (tab[0], then per higher byte its entry and its bond).
#pragma unroll 4
            for (unsigned s = 4u * threadIdx.x; s < ns; s += 4u * BT_THREADS) {
                const float4 c4 = *reinterpret_cast<const float4*>(C + s);
                const float4 t0 = *reinterpret_cast<const float4*>(&tab[0][s & 255u]);
                float w0 = t0.x, w1 = t0.y, w2 = t0.z, w3 = t0.w;
                const unsigned x = s ^ (s >> 1);
                for (int m = 1; m < nchunk; ++m) {
                    const float tm = tab[m][(s >> (8 * m)) & 255u];
                    const float bd = ((x >> (8 * m - 1)) & 1u) ? -kacc[8 * m - 1] : kacc[8 * m - 1];
                    w0 += tm; w1 += tm; w2 += tm; w3 += tm;
                    w0 += bd; w1 += bd; w2 += bd; w3 += bd;
                }
                const float v0 = c4.x + w0, v1 = c4.y + w1, v2 = c4.z + w2, v3 = c4.w + w3;
                if (v0 > bv) { bv = v0; b32 = s; }
                if (v1 > bv) { bv = v1; b32 = s + 1; }
                if (v2 > bv) { bv = v2; b32 = s + 2; }
                if (v3 > bv) { bv = v3; b32 = s + 3; }
            }
        } else {
            for (unsigned s = threadIdx.x; s < ns; s += BT_THREADS) visit(C[s], s);
        }
        if (b32 != 0xffffffffu) bs = b32;
        for (int o = 16; o; o >>= 1) {
            float v2 = __shfl_xor_sync(0xffffffffu, bv, o);
            unsigned long long s2 = __shfl_xor_sync(0xffffffffu, bs, o);
            argmax_combine(bv, bs, v2, s2);
        }
        if ((threadIdx.x & 31) == 0) { rv[threadIdx.x >> 5] = bv; rs[threadIdx.x >> 5] = bs; }
        __syncthreads();
        if (threadIdx.x == 0) {
            for (int w = 1; w < BT_THREADS / 32; ++w) argmax_combine(bv, bs, rv[w], rs[w]);
            s_next = bs;
            p.s_out[inst] = bs;
            if (!has_next) p.v_out[inst] = bv;
        }
        __syncthreads();
        if (threadIdx.x < L)
            p.sigma[(inst * L + r) * L + threadIdx.x] = ((s_next >> threadIdx.x) & 1ull) ? -1 : 1;
    }
}

// ---- S0 of the generic path: conjugated gate constants and the coefficients of A_{L-1} -------------
struct GenericPrepParams {
    int col_off;                   // Z3: 1 = Op.c is a stored digit, lattice column = c + 1; Op.c = VCOL is column 0
    int q, L, n_ops;
    const Op* ops;                 // [n_ops] gates in execution order
    const float* Jh; const float* Jv; const float* h;   // device couplings, per instance
    float* gate_k;                 // [inst][n_ops][8]
    float* fin;                    // [inst][2 * GMAX_L]
};

__global__ void __launch_bounds__(256) generic_prep_kernel(const GenericPrepParams p) {
    const unsigned long long inst = blockIdx.y;
    const int L = p.L;
    const float* Jh = p.Jh + inst * (unsigned long long)(L * (L - 1));
    const float* Jv = p.Jv + inst * (unsigned long long)((L - 1) * L);
    const float* hh = p.h ? p.h + inst * (unsigned long long)(L * L) : nullptr;
    const long idx = (long)blockIdx.x * blockDim.x + threadIdx.x;
    auto Hacc = [&](int R, int c) { double s = 0; if (hh) for (int r = 0; r < R; ++r) s += (double)hh[r * L + c]; return s; };
    auto Kacc = [&](int R, int c) { double s = 0; if (c < 0 || c >= L - 1) return s; for (int r = 0; r < R; ++r) s += (double)Jh[r * (L - 1) + c]; return s; };
    if (idx < p.n_ops) {
        const Op op = p.ops[idx];
        const int r = op.row, c = op.c == VCOL ? 0 : op.c + p.col_off;          // lattice column
        float* out = p.gate_k + (inst * p.n_ops + idx) * 8;
        const double J = (double)Jv[(r - 1) * L + c], Kl = Kacc(r, c - 1), Kr = Kacc(r, c);
        if (p.q == 2) {
            const double m = -2.0 * J, H = Hacc(r, c);
            for (int nl = 0; nl < 2; ++nl)
                for (int nr = 0; nr < 2; ++nr) {
                    const double rho = H + (nl ? -Kl : Kl) + (nr ? -Kr : Kr);
                    out[nl * 2 + nr] = (float)(m - 2.0 * rho);          // ka
                    out[4 + nl * 2 + nr] = (float)(m + 2.0 * rho);      // kb
                }
        } else {
            out[0] = (float)J; out[1] = (float)Kl; out[2] = (float)Kr;
            for (int i = 3; i < 8; ++i) out[i] = 0.f;
        }
    }
    if (idx < 2 * GMAX_L) {
        float* out = p.fin + inst * (2 * GMAX_L);
        const int c = (int)(idx % GMAX_L) + p.col_off;                          // tables are per stored digit
        if (idx < GMAX_L) out[idx] = p.col_off ? (idx == 0 ? (float)Kacc(L, 0) : 0.f)   // Z3: slot 0 = the bond column 0 - column 1
                                               : (c < L ? (float)Hacc(L, c) : 0.f);
        else out[idx] = c < L - 1 ? (float)Kacc(L, c) : 0.f;
    }
}

}  // namespace ttn
