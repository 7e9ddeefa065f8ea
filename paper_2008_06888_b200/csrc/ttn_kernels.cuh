// ttn_kernels.cuh -- device side of the tropical transfer sweep, generic ("v1") path.
//
// One launch of pass_kernel = one HBM pass over the q^L state: each
// CTA stages one tile (digits [0,lo) U [a,b) of the state index) in shared memory, runs the
// pass's op list on it -- max-plus gates (A2) PAPER.md:242 / the 3x3 Potts gate of App. C
// PAPER.md:296 as butterflies over the gate's digit, diagonal terms (A3), (A4)
// PAPER.md:247-252 as elementwise adds -- and writes it back in place ("all
// operations should be performed inplace").  The first pass is write-only (initial state
// (0,0)^{(x)L}), the last is read-only and fuses the final (+)-reduction.
//
// Semirings: Tropical<f32>: x (+) y = max, x (.) y = x + y (Eq. (2)
// PAPER.md:57); CountingTropical<f32,f64>: Eq. (4), counts summed on exact ties.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>
#include "planner.h"

namespace ttn {

struct PassParams {
    int L, T, lo, a, b;
    unsigned long long P_lo, P_a, P_mid, P_b;   // q^lo, q^a, q^(a-lo), q^b
    unsigned int n_tile;                          // q^T elements per tile
    unsigned long long tiles_per_inst;            // q^(L-T)
    const float* src_x; float* dst_x;             // instance 0 base pointers
    const double* src_n; double* dst_n;           // counting only
    unsigned long long src_stride, dst_stride;    // elements between instances
    const Op* ops; int n_ops;
    const float* Jh; const float* Jv; const float* h;   // device, per instance; h may be null
    int flags;
    float* part_x; double* part_n;                // [inst][tile] partial reductions
};

// ---------------------------------------------------------------------------------------------
template <int Q> struct Radix;
template <> struct Radix<2> {
    __device__ static __forceinline__ unsigned digit(unsigned long long s, int c) { return (unsigned)(s >> c) & 1u; }
};
template <> struct Radix<3> {
    __device__ static __forceinline__ unsigned digit(unsigned long long s, int c) {
        const unsigned p3[21] = {1u, 3u, 9u, 27u, 81u, 243u, 729u, 2187u, 6561u, 19683u, 59049u, 177147u,
                                 531441u, 1594323u, 4782969u, 14348907u, 43046721u, 129140163u,
                                 387420489u, 1162261467u, 3486784401u};
        return ((unsigned)s / p3[c]) % 3u;       // Potts index fits 32 bits (L <= 20)
    }
};

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
    if (COUNT) {
        if (cx > x) { x = cx; n = cn; }
        else if (cx == x) { n += cn; }
    } else {
        x = fmaxf(x, cx);
    }
}

template <int Q, bool COUNT>
__global__ void __launch_bounds__(512) pass_kernel(const PassParams p) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double* sn = reinterpret_cast<double*>(smem_raw);                       // [n_tile] if COUNT
    float* sx = reinterpret_cast<float*>(smem_raw + (COUNT ? (size_t)p.n_tile * 8 : 0));
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
    __syncthreads();

    const float* Jh = p.Jh + inst * (unsigned long long)(p.L * (p.L - 1));
    const float* Jv = p.Jv + inst * (unsigned long long)((p.L - 1) * p.L);
    const float* hh = p.h ? p.h + inst * (unsigned long long)(p.L * p.L) : nullptr;

    // ---- op list ------------------------------------------------------------------------------
    for (int k = 0; k < p.n_ops; ++k) {
        const Op op = p.ops[k];
        if (op.type == OP_GATE) {
            const float J = Jv[(op.row - 1) * p.L + op.c];
            // stride of the gate's digit inside the tile
            unsigned st = 1;
            for (int i = 0; i < op.pos; ++i) st *= Q;
            const unsigned ngrp = N / Q;
            for (unsigned g = threadIdx.x; g < ngrp; g += blockDim.x) {
                unsigned i0 = (g / st) * (st * Q) + (g % st);
                if (Q == 2) {
                    // (A2): new[b'] = max_b(old[b] + J s(b) s(b')) = J + max(old[b'], old[1-b'] - 2J);
                    // the common +J is deferred to a per-instance scalar (see api: defer).
                    const float m = -2.f * J;
                    float xa = sx[i0], xb = sx[i0 + st];
                    float ca = xb + m, cb = xa + m;
                    if (COUNT) {
                        double na = sn[i0], nb = sn[i0 + st];
                        float ya = xa; double ma = na; oplus<true>(ya, ma, ca, nb);
                        float yb = xb; double mb = nb; oplus<true>(yb, mb, cb, na);
                        sx[i0] = ya; sx[i0 + st] = yb; sn[i0] = ma; sn[i0 + st] = mb;
                    } else {
                        sx[i0] = fmaxf(xa, ca); sx[i0 + st] = fmaxf(xb, cb);
                    }
                } else {
                    // Potts: new[t'] = max_t(old[t] + J delta(t,t'))
                    float x0 = sx[i0], x1 = sx[i0 + st], x2 = sx[i0 + 2 * st];
                    if (COUNT) {
                        double n0 = sn[i0], n1 = sn[i0 + st], n2 = sn[i0 + 2 * st];
                        float y0 = x0 + J; double m0 = n0; oplus<true>(y0, m0, x1, n1); oplus<true>(y0, m0, x2, n2);
                        float y1 = x1 + J; double m1 = n1; oplus<true>(y1, m1, x0, n0); oplus<true>(y1, m1, x2, n2);
                        float y2 = x2 + J; double m2 = n2; oplus<true>(y2, m2, x0, n0); oplus<true>(y2, m2, x1, n1);
                        sx[i0] = y0; sx[i0 + st] = y1; sx[i0 + 2 * st] = y2;
                        sn[i0] = m0; sn[i0 + st] = m1; sn[i0 + 2 * st] = m2;
                    } else {
                        sx[i0] = fmaxf(x0 + J, fmaxf(x1, x2));
                        sx[i0 + st] = fmaxf(x1 + J, fmaxf(x0, x2));
                        sx[i0 + 2 * st] = fmaxf(x2 + J, fmaxf(x0, x1));
                    }
                }
            }
            __syncthreads();
        } else {
            // a run of diagonal terms: one sweep over the tile applies them all, in list order
            int k2 = k;
            while (k2 + 1 < p.n_ops && p.ops[k2 + 1].type != OP_GATE) ++k2;
            for (unsigned t = threadIdx.x; t < N; t += blockDim.x) {
                unsigned long long s = base + (unsigned long long)(t % plo) + (unsigned long long)(t / plo) * p.P_a;
                float v = sx[t];
                for (int j = k; j <= k2; ++j) {
                    const Op o = p.ops[j];
                    if (o.type == OP_DH) {
                        if (Q == 2 && hh) {
                            float hv = hh[o.row * p.L + o.c];
                            v += Radix<Q>::digit(s, o.c) ? -hv : hv;
                        }
                    } else {
                        float Jc = Jh[o.row * (p.L - 1) + o.c];
                        unsigned d0 = Radix<Q>::digit(s, o.c), d1 = Radix<Q>::digit(s, o.c + 1);
                        if (Q == 2) v += (d0 == d1) ? Jc : -Jc;
                        else v += (d0 == d1) ? Jc : 0.f;
                    }
                }
                sx[t] = v;
            }
            k = k2;
            __syncthreads();
        }
    }

    // ---- store, or reduce ------------------------------------------------------------------
    if (p.flags & PASS_REDUCE) {
        float mx = -INFINITY;
        for (unsigned t = threadIdx.x; t < N; t += blockDim.x) mx = fmaxf(mx, sx[t]);
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
// backtracking"): s_{L-1} = argmax_s C_{L-1}[s];  s_r = argmax_s ( C_r[s] + sum_c Jv[r][c]
// sigma_c(s) sigma_c(s_{r+1}) ).  Lowest index wins ties (footnote [49] PAPER.md:201).
struct ArgmaxParams {
    int L, r, has_next, nblk;
    unsigned long long NS;
    const float* C;                     // checkpoint C_r of instance 0
    unsigned long long c_stride;        // elements between instances
    const float* Jv;                    // device couplings (per instance)
    const unsigned long long* s_next;   // [batch] state of row r+1 (if has_next)
    float* part_v; unsigned long long* part_s;   // [batch][nblk]
    unsigned long long* s_out;          // [batch]
    float* v_out;                       // [batch] max value (written when !has_next)
    signed char* sigma;                 // [batch][L][L]
};

__device__ __forceinline__ void argmax_combine(float& v, unsigned long long& s, float v2, unsigned long long s2) {
    if (v2 > v || (v2 == v && s2 < s)) { v = v2; s = s2; }
}

__global__ void __launch_bounds__(256) argmax_partial_kernel(const ArgmaxParams p) {
    const unsigned long long inst = blockIdx.y;
    __shared__ float jsig[64];
    if (threadIdx.x < p.L) {
        float j = 0.f;
        if (p.has_next) {
            j = p.Jv[inst * (unsigned long long)((p.L - 1) * p.L) + p.r * p.L + threadIdx.x];
            if ((p.s_next[inst] >> threadIdx.x) & 1ull) j = -j;
        }
        jsig[threadIdx.x] = j;
    }
    __syncthreads();
    const float* C = p.C + inst * p.c_stride;
    float bv = -INFINITY; unsigned long long bs = ~0ull;
    for (unsigned long long s = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; s < p.NS;
         s += (unsigned long long)gridDim.x * blockDim.x) {
        float w = 0.f;
        if (p.has_next)
            for (int c = 0; c < p.L; ++c) w += ((s >> c) & 1ull) ? -jsig[c] : jsig[c];
        argmax_combine(bv, bs, C[s] + w, s);
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

}  // namespace ttn
