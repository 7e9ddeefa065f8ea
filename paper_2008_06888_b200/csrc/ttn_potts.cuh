// ttn_potts.cuh -- q = 3 Potts tile kernel with register-blocked gates.
//
// Same pass structure, tile geometry, diagonal frame and gate constants as the generic kernel of
// ttn_kernels.cuh (one CTA stages the 3^T-element tile [0,lo) U [a,b) in shared memory, applies
// the pass's gates, writes it back in place), but the gates of App. C PAPER.md:296 are applied in
// BLOCKS of up to three adjacent columns c, c+1, c+2 of one lattice row (planner.h
// mark_gate_blocks): a thread pulls the 3^NB elements that differ in those NB digits into
// registers, applies the NB gates to them (3^(NB-1) triples each) and puts them back -- one
// shared-memory round trip per NB gates, the index arithmetic paid once.
//
// Conjugation inside a block.  In the diagonal frame the gate on column c is
// A^{-1} G(c) A with A = A_{r-1} (ttn_kernels.cuh header); only A's bonds (c-1,c) and (c,c+1)
// matter.  Gates of one row share A, so  G''(c) G''(c+1) G''(c+2) = A^{-1} G(c) G(c+1) G(c+2) A:
// the bonds INSIDE the block are added to the registers once before the gates and removed once
// after them (elements whose two digits agree: + K, App. C PAPER.md:296 delta form); the bond to
// the left of the first column wraps only the first gate, the bond to the right of the last
// column only the last gate (R(t) = K delta(t, neighbour digit), neighbour digit from the
// element's own index).
//
// Counting (Eq. (4)): new n = sum of the n_t of the exact maximisers, formed as FP64
// multiply-adds with 0/1 indicators.
//
#pragma once
#include "ttn_kernels.cuh"

namespace ttn {

// m += n  if  c == best: FSETP + SEL of the indicator's high word + DFMA (ptxas turns a predicated
// DADD into two FSELs of the addend, which costs the alu pipe one more slot per candidate)
__device__ __forceinline__ void add_if_eq(double& m, float c, float best, double n) { m = fma(n, ind01(c == best), m); }

// One 3x3 gate on the triple (x0,x1,x2): y_t = x_t + R_t, new_t' = max_t(y_t + J delta(t,t')) - R_t'.
// HAS_R = false: R = 0 (both bonds of this column are handled by the block).
template <bool COUNT, bool HAS_R>
__device__ __forceinline__ void potts_gate3(float& x0, float& x1, float& x2, double& n0, double& n1, double& n2,
                                            float J, float R0, float R1, float R2) {
    const float y0 = HAS_R ? x0 + R0 : x0, y1 = HAS_R ? x1 + R1 : x1, y2 = HAS_R ? x2 + R2 : x2;
    const float j0 = y0 + J, j1 = y1 + J, j2 = y2 + J;
    const float b0 = max3(j0, y1, y2), b1 = max3(y0, j1, y2), b2 = max3(y0, y1, j2);
    if (COUNT) {
        double m0 = 0.0, m1 = 0.0, m2 = 0.0;
        add_if_eq(m0, j0, b0, n0); add_if_eq(m0, y1, b0, n1); add_if_eq(m0, y2, b0, n2);
        add_if_eq(m1, y0, b1, n0); add_if_eq(m1, j1, b1, n1); add_if_eq(m1, y2, b1, n2);
        add_if_eq(m2, y0, b2, n0); add_if_eq(m2, y1, b2, n1); add_if_eq(m2, j2, b2, n2);
        n0 = m0; n1 = m1; n2 = m2;
    }
    x0 = HAS_R ? b0 - R0 : b0; x1 = HAS_R ? b1 - R1 : b1; x2 = HAS_R ? b2 - R2 : b2;
}

// digit j (0..NB-1) of the register index e = d0 + 3 d1 + 9 d2
__device__ __forceinline__ constexpr int pdig(int e, int j) { return j == 0 ? e % 3 : (j == 1 ? (e / 3) % 3 : e / 9); }
__device__ __forceinline__ constexpr int ppow3(int j) { return j == 0 ? 1 : (j == 1 ? 3 : 9); }

// aux: x = 3^pos, y = magic(3^pos), z = magic(3^(pos-1)),
//      w = l_in | r_in << 1 | nb << 2 | (s_dig slot of the left outer column) << 8 | (slot of the right one) << 16
// gk:  this block's gate constants in shared memory, one float4 per gate: (Jv, Kl, Kr, -)
template <int NB, bool COUNT>
__device__ __forceinline__ void potts_block(float* __restrict__ sx, double* __restrict__ sn, unsigned N,
                                            const uint4 aux, const float4* __restrict__ gk, const int* s_dig) {
    constexpr int E = NB == 1 ? 3 : (NB == 2 ? 9 : 27);
    const unsigned st = aux.x, m_st = aux.y, m_stq = aux.z;
    const bool l_in = aux.w & 1u, r_in = (aux.w >> 1) & 1u;
    const int dl_out = s_dig[(aux.w >> 8) & 255u], dr_out = s_dig[(aux.w >> 16) & 255u];
    float J[NB], KB[NB];                               // KB[j] = bond to the right of block column j
#pragma unroll
    for (int j = 0; j < NB; ++j) { J[j] = gk[j].x; KB[j] = gk[j].z; }
    const float Kl = gk[0].y, Kr = KB[NB - 1];
    const unsigned ngrp = N / E;
    for (unsigned g = threadIdx.x; g < ngrp; g += blockDim.x) {
        const unsigned hi = st == 1 ? g : fastdiv(g, m_st), lo = g - hi * st;
        const int dl = l_in ? (int)(st == 3 ? lo : fastdiv(lo, m_stq)) : dl_out;
        const int dr = r_in ? (int)(hi % 3u) : dr_out;
        const unsigned i0 = hi * (st * E) + lo;
        float x[E]; double n[E];
#pragma unroll
        for (int e = 0; e < E; ++e) { x[e] = sx[i0 + e * st]; if (COUNT) n[e] = sn[i0 + e * st]; else n[e] = 0.0; }
        // bonds inside the block
#pragma unroll
        for (int j = 0; j + 1 < NB; ++j)
#pragma unroll
            for (int e = 0; e < E; ++e) if (pdig(e, j) == pdig(e, j + 1)) x[e] += KB[j];
        const float RL0 = dl == 0 ? Kl : 0.f, RL1 = dl == 1 ? Kl : 0.f, RL2 = dl == 2 ? Kl : 0.f;
        const float RR0 = dr == 0 ? Kr : 0.f, RR1 = dr == 1 ? Kr : 0.f, RR2 = dr == 2 ? Kr : 0.f;
#pragma unroll
        for (int j = 0; j < NB; ++j) {
            const int s = ppow3(j);
#pragma unroll
            for (int e = 0; e < E; ++e) {
                if (pdig(e, j) != 0) continue;                       // e = the triple's t = 0 element
                if (NB == 1)
                    potts_gate3<COUNT, true>(x[e], x[e + s], x[e + 2 * s], n[e], n[e + s], n[e + 2 * s], J[j],
                                             RL0 + RR0, RL1 + RR1, RL2 + RR2);
                else if (j == 0)
                    potts_gate3<COUNT, true>(x[e], x[e + s], x[e + 2 * s], n[e], n[e + s], n[e + 2 * s], J[j], RL0, RL1, RL2);
                else if (j == NB - 1)
                    potts_gate3<COUNT, true>(x[e], x[e + s], x[e + 2 * s], n[e], n[e + s], n[e + 2 * s], J[j], RR0, RR1, RR2);
                else
                    potts_gate3<COUNT, false>(x[e], x[e + s], x[e + 2 * s], n[e], n[e + s], n[e + 2 * s], J[j], 0.f, 0.f, 0.f);
            }
        }
#pragma unroll
        for (int j = 0; j + 1 < NB; ++j)
#pragma unroll
            for (int e = 0; e < E; ++e) if (pdig(e, j) == pdig(e, j + 1)) x[e] -= KB[j];
        // the addresses are formed again for the stores (an opaque copy of i0) so that the 3^NB
        // load addresses do not stay live across the gates
        unsigned j0 = i0;
        asm volatile("" : "+r"(j0));
#pragma unroll
        for (int e = 0; e < E; ++e) { sx[j0 + e * st] = x[e]; if (COUNT) sn[j0 + e * st] = n[e]; }
    }
}


__device__ __forceinline__ void cp_async4(void* smem, const void* g) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" :: "r"((unsigned)__cvta_generic_to_shared(smem)), "l"(g) : "memory");
}
__device__ __forceinline__ void cp_async8(void* smem, const void* g) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" :: "r"((unsigned)__cvta_generic_to_shared(smem)), "l"(g) : "memory");
}

constexpr int POTTS_THREADS = 256;       // energy: 3^9 tile = 729 groups of 27 (blocks of 3 gates)
constexpr int POTTS_THREADS_COUNT = 384; // counting: 3^8 tile = 729 groups of 9 (blocks of 2 gates; 27 (x, n) pairs do not fit 128 registers)
constexpr int POTTS_MAX_NB_COUNT = 2;
constexpr int POTTS_MAX_OPS = 256;       // gates of one pass (host checks)
__host__ __device__ inline size_t potts_buf_bytes(unsigned n_tile, bool count) { return ((size_t)n_tile * (count ? 12 : 4) + 15) / 16 * 16; }

// first element of global tile `gtile` (instance-relative) and its instance
struct PottsTile { unsigned inst, base; };
__device__ __forceinline__ PottsTile potts_tile(const PassParams& p, unsigned gtile) {
    const unsigned tpi = (unsigned)p.tiles_per_inst, pmid = (unsigned)p.P_mid;
    PottsTile t;
    t.inst = gtile / tpi;
    const unsigned tile = gtile - t.inst * tpi, hi = tile / pmid;
    t.base = (tile - hi * pmid) * (unsigned)p.P_lo + hi * (unsigned)p.P_b;       // 3^L < 2^32 for L <= 20
    return t;
}

// Persistent: two CTAs per SM, each loads (cp.async), computes and stores one tile after the other;
// tile t goes to CTA t mod gridDim, so the CTAs running at any moment work on neighbouring tiles
// (their rows continue one another in memory).  Measured alternatives that were slower and are
// not kept: one double-buffered CTA per SM prefetching the next tile, a contiguous range of tiles
// per CTA, a start-up stagger between the two residents of an SM (profiles/r01j.md).
template <bool COUNT, int THREADS>
__global__ void __launch_bounds__(THREADS, 2) potts_pass_kernel(const PassParams p, const unsigned total_tiles) {
    constexpr int Q = 3;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const unsigned N = p.n_tile;
    double* sn = reinterpret_cast<double*>(smem_raw);                       // [N] if COUNT
    float* sx = reinterpret_cast<float*>(smem_raw + (COUNT ? (size_t)N * 8 : 0));
    __shared__ int s_dig[GMAX_L + 1];        // digits of the tile's base index; slot GMAX_L = 0 ("no such column")
    __shared__ float s_fin[GMAX_L];          // K_c of A_{L-1} (REDUCE pass)
    __shared__ float s_aout;                 // part of A_{L-1} that only involves columns outside the tile
    __shared__ float s_tabA[81], s_tabB[243]; // A_{L-1} over the low 4 / the other <= 5 tile digits (T <= 9)
    __shared__ uint4 s_aux[POTTS_MAX_OPS];   // per gate (block leaders are the ones used)
    __shared__ float4 s_gk[POTTS_MAX_OPS];   // gate constants of the current instance
    __shared__ unsigned char s_list[POTTS_MAX_OPS];   // op index of every block leader
    __shared__ int s_nblk;
    __shared__ float red_x[THREADS / 32];
    __shared__ double red_n[THREADS / 32];
    const unsigned plo = (unsigned)p.P_lo, m_plo = fastdiv_magic(plo);      // rows of plo contiguous elements
    const unsigned pa = (unsigned)p.P_a;
    const bool init = p.flags & PASS_INIT, reduce = p.flags & PASS_REDUCE;

    // per-gate index constants that do not depend on the tile
    for (int i = threadIdx.x; i < p.n_ops; i += THREADS) {
        const Op o = p.ops[i];
        const int nb = o.nb > 0 ? o.nb : 1;
        unsigned s_ = 1;
        for (int j = 0; j < o.pos; ++j) s_ *= Q;
        const unsigned sq = o.pos > 0 ? s_ / Q : 1;
        const int cl = o.c - 1, cr = o.c + nb;                 // the block's outer neighbour columns
        const bool li = o.pos > 0 && tile_col(p, o.pos - 1) == cl;
        const bool ri = o.pos + nb < p.T && tile_col(p, o.pos + nb) == cr;
        const unsigned sl = cl >= 0 ? cl : GMAX_L, sr = cr < p.L ? cr : GMAX_L;
        s_aux[i] = make_uint4(s_, fastdiv_magic(s_), fastdiv_magic(sq),
                              (unsigned)li | ((unsigned)ri << 1) | ((unsigned)o.nb << 2) | (sl << 8) | (sr << 16));
    }
    if (threadIdx.x == 0) {
        s_dig[GMAX_L] = 0;
        int nblk = 0;
        for (int i = 0; i < p.n_ops; ++i) if (p.ops[i].nb) s_list[nblk++] = (unsigned char)i;
        s_nblk = nblk;
    }

    unsigned last_inst = 0xffffffffu;
    for (unsigned gtile = blockIdx.x; gtile < total_tiles; gtile += gridDim.x) {
        const PottsTile tl = potts_tile(p, gtile);
        __syncthreads();                     // everyone is done with the previous tile
        // ---- load (or initialise to the semiring one) ----------------------------------------
        if (init) {
            for (unsigned e = threadIdx.x; e < N; e += THREADS) { sx[e] = 0.f; if (COUNT) sn[e] = 1.0; }
        } else {
            const float* gx = p.src_x + (unsigned long long)tl.inst * p.src_stride + tl.base;
            const double* gn = COUNT ? p.src_n + (unsigned long long)tl.inst * p.src_stride + tl.base : nullptr;
            for (unsigned e = threadIdx.x; e < N; e += THREADS) {
                const unsigned row = plo == 1 ? e : fastdiv(e, m_plo);
                const unsigned off = (e - row * plo) + row * pa;
                cp_async4(sx + e, gx + off);
                if (COUNT) cp_async8(sn + e, gn + off);
            }
        }
        for (int i = threadIdx.x; i < p.L; i += THREADS) {   // digit c of the base index (0 for the tile's own columns)
            unsigned pw = 1;
            for (int c = 0; c < i; ++c) pw *= Q;
            s_dig[i] = (int)((tl.base / pw) % Q);
        }
        if (tl.inst != last_inst) {
            if (reduce)
                for (int i = threadIdx.x; i < GMAX_L; i += THREADS) s_fin[i] = p.fin[(size_t)tl.inst * (2 * GMAX_L) + GMAX_L + i];
            const float4* GK = reinterpret_cast<const float4*>(p.gate_k + (unsigned long long)tl.inst * p.gate_inst_stride);
            for (int i = threadIdx.x; i < p.n_ops; i += THREADS) s_gk[i] = GK[2 * i];
            last_inst = tl.inst;
        }
        asm volatile("cp.async.wait_all;" ::: "memory");
        __syncthreads();

        // ---- gate blocks -----------------------------------------------------------------------
        const int nblk = s_nblk;
        for (int j = 0; j < nblk; ++j) {
            const int k = s_list[j];
            const uint4 aux = s_aux[k];
            const int nb = (int)((aux.w >> 2) & 3u);
            const float4* gk = s_gk + k;
            if (!COUNT && nb == 3) potts_block<3, COUNT>(sx, sn, N, aux, gk, s_dig);   // counting: blocks of <= 2
            else if (nb == 2) potts_block<2, COUNT>(sx, sn, N, aux, gk, s_dig);
            else potts_block<1, COUNT>(sx, sn, N, aux, gk, s_dig);
            __syncthreads();
        }

        // ---- store, or multiply by A_{L-1}(s) and reduce ------------------------------------------
        if (reduce) {
            const float* K = s_fin;
            if (threadIdx.x == 0) {              // bonds whose columns both lie outside the tile
                float acc = 0.f;
                for (int c = 0; c + 1 < p.L; ++c) {
                    const bool in_c = c < p.lo || (c >= p.a && c < p.b);
                    const bool in_n = c + 1 < p.lo || (c + 1 >= p.a && c + 1 < p.b);
                    if (!in_c && !in_n) acc += diag2<Q>(K[c], s_dig[c], s_dig[c + 1]);
                }
                s_aout = acc;
            }
            __syncthreads();
            // A_{L-1}(s) restricted to the tile = table over the low (<= 4) tile digits + table over
            // the other (<= 5) digits + the one bond between the two groups
            const int GA = p.T < 4 ? p.T : 4;
            unsigned NA = 1;
            for (int i = 0; i < GA; ++i) NA *= Q;
            const unsigned NBH = N / NA, m_na = fastdiv_magic(NA);
            auto terms = [&](unsigned idx, int pos0, int pos1) {
                float acc = 0.f;
                unsigned rest = idx;
                int dprev = 0, cprev = -2;
                for (int pos = pos0; pos < pos1; ++pos) {
                    const int d = (int)(rest % Q); rest /= Q;
                    const int c = tile_col(p, pos);
                    if (c > 0) {
                        if (cprev == c - 1) acc += diag2<Q>(K[c - 1], dprev, d);                 // left neighbour in this group
                        else if (!(pos > 0 && tile_col(p, pos - 1) == c - 1)) acc += diag2<Q>(K[c - 1], s_dig[c - 1], d);   // outside the tile
                    }                                                                            // else: the bond between the groups
                    const bool right_in = pos + 1 < p.T && tile_col(p, pos + 1) == c + 1;
                    if (c + 1 < p.L && !right_in) acc += diag2<Q>(K[c], d, s_dig[c + 1]);
                    dprev = d; cprev = c;
                }
                return acc;
            };
            for (unsigned i = threadIdx.x; i < NA; i += THREADS) s_tabA[i] = terms(i, 0, GA);
            for (unsigned i = threadIdx.x; i < NBH; i += THREADS) s_tabB[i] = terms(i, GA, p.T);
            const bool has_x = GA < p.T && tile_col(p, GA) == tile_col(p, GA - 1) + 1;
            const float Kx = has_x ? K[tile_col(p, GA - 1)] : 0.f;
            __syncthreads();
            float mx = -INFINITY;
            for (unsigned e = threadIdx.x; e < N; e += THREADS) {
                const unsigned hi = NA == N ? 0u : fastdiv(e, m_na), lo = e - hi * NA;
                float acc = s_aout + s_tabA[lo] + s_tabB[hi];
                if (lo / (NA / Q) == hi % Q) acc += Kx;
                const float val = sx[e] + acc;
                sx[e] = val;
                mx = fmaxf(mx, val);
            }
            mx = warp_max(mx);
            if ((threadIdx.x & 31) == 0) red_x[threadIdx.x >> 5] = mx;
            __syncthreads();
            float bm = red_x[0];
            for (int w = 1; w < THREADS / 32; ++w) bm = fmaxf(bm, red_x[w]);
            double cnt = 0.0;
            if (COUNT) {
                for (unsigned e = threadIdx.x; e < N; e += THREADS) if (sx[e] == bm) cnt += sn[e];
                cnt = warp_sum(cnt);
                if ((threadIdx.x & 31) == 0) red_n[threadIdx.x >> 5] = cnt;
                __syncthreads();
            }
            if (threadIdx.x == 0) {
                p.part_x[gtile] = bm;
                if (COUNT) {
                    double tot = 0.0;
                    for (int w = 0; w < THREADS / 32; ++w) tot += red_n[w];
                    p.part_n[gtile] = tot;
                }
            }
        } else {
            float* gx = p.dst_x + (unsigned long long)tl.inst * p.dst_stride + tl.base;
            double* gn = COUNT ? p.dst_n + (unsigned long long)tl.inst * p.dst_stride + tl.base : nullptr;
            for (unsigned e = threadIdx.x; e < N; e += THREADS) {
                const unsigned row = plo == 1 ? e : fastdiv(e, m_plo);
                const unsigned off = (e - row * plo) + row * pa;
                gx[off] = sx[e];
                if (COUNT) gn[off] = sn[e];
            }
        }
    }
}

}  // namespace ttn
