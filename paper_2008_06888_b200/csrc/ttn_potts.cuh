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
// s_dig: [member][GMAX_L + 1] digits of the base index of every tile the CTA holds (one, or the three of
// a rotation orbit: N = 3 Nm elements, member = element index / Nm); gpm = groups per member (0: one member)
template <int NB, bool COUNT>
__device__ __forceinline__ void potts_block(float* __restrict__ sx, double* __restrict__ sn, unsigned N,
                                            const uint4 aux, const float4* __restrict__ gk,
                                            const int (*s_dig)[GMAX_L + 1], const unsigned gpm) {
    constexpr int E = NB == 1 ? 3 : (NB == 2 ? 9 : 27);
    const unsigned st = aux.x, m_st = aux.y, m_stq = aux.z;
    const bool l_in = aux.w & 1u, r_in = (aux.w >> 1) & 1u;
    const unsigned slot_l = (aux.w >> 8) & 255u, slot_r = (aux.w >> 16) & 255u;
    const unsigned m_gpm = fastdiv_magic(gpm);
    float J[NB], KB[NB];                               // KB[j] = bond to the right of block column j
#pragma unroll
    for (int j = 0; j < NB; ++j) { J[j] = gk[j].x; KB[j] = gk[j].z; }
    const float Kl = gk[0].y, Kr = KB[NB - 1];
    const unsigned ngrp = N / E;
    for (unsigned g = threadIdx.x; g < ngrp; g += blockDim.x) {
        const unsigned hi = st == 1 ? g : fastdiv(g, m_st), lo = g - hi * st;
        const unsigned mem = gpm == 0u ? 0u : (gpm == 1u ? g : fastdiv(g, m_gpm));
        const int dl = l_in ? (int)(st == 3 ? lo : fastdiv(lo, m_stq)) : s_dig[mem][slot_l];
        const int dr = r_in ? (int)(hi % 3u) : s_dig[mem][slot_r];
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

// ---- Z3 reduction (planner.h "COLOUR-ROTATION (Z3) REDUCTION") --------------------------------------------
// The CTA holds the three member tiles of a rotation orbit: member o = every outside digit of member 0
// plus o (mod 3); element (o, e) of the CTA buffer is local index e of member o.  The gate on column 0
// acts on x_k = W[k, rest] = H[rho^-k rest]: for rest = (member 0, e) these are (0, e), (2, r1(e)), (1, r2(e))
// with r1 = "every local digit minus 1", r2 = r1 o r1 (table s_rot).  Every element of the buffer is in
// exactly one such triple.  R(t) = K_0 delta(t, t_1), t_1 = the column-1 digit (digit 0) of rest.
template <bool COUNT>
__device__ __forceinline__ void potts_vgate(float* __restrict__ sx, double* __restrict__ sn, const unsigned Nm,
                                            const float4 gk, const unsigned short* __restrict__ s_rot,
                                            const bool d0_in_tile, const int d0_out) {
    const float J = gk.x, K0 = gk.z;
    for (unsigned e = threadIdx.x; e < Nm; e += blockDim.x) {
        const unsigned e1 = s_rot[e], e2 = s_rot[e1];
        const unsigned i0 = e, i1 = 2u * Nm + e1, i2 = Nm + e2;
        const int t1 = d0_in_tile ? (int)(e % 3u) : d0_out;
        float x0 = sx[i0], x1 = sx[i1], x2 = sx[i2];
        double n0 = 0.0, n1 = 0.0, n2 = 0.0;
        if (COUNT) { n0 = sn[i0]; n1 = sn[i1]; n2 = sn[i2]; }
        potts_gate3<COUNT, true>(x0, x1, x2, n0, n1, n2, J, t1 == 0 ? K0 : 0.f, t1 == 1 ? K0 : 0.f, t1 == 2 ? K0 : 0.f);
        sx[i0] = x0; sx[i1] = x1; sx[i2] = x2;
        if (COUNT) { sn[i0] = n0; sn[i1] = n1; sn[i2] = n2; }
    }
}

constexpr int POTTS_THREADS = 256;       // energy: 3^9 tile = 729 groups of 27 (blocks of 3 gates)
constexpr int POTTS_THREADS_COUNT = 384; // counting: 3^8 tile = 729 groups of 9 (blocks of 2 gates; 27 (x, n) pairs do not fit 128 registers)
constexpr int POTTS_MAX_NB_COUNT = 2;
constexpr int POTTS_MAX_OPS = 256;       // gates of one pass (host checks)
__host__ __device__ inline size_t potts_buf_bytes(unsigned n_tile, bool count) { return ((size_t)n_tile * (count ? 12 : 4) + 15) / 16 * 16; }
// Z3: three member tiles + the rotation table (u16 per local index)
__host__ __device__ inline size_t potts_z3_bytes(unsigned n_member, bool count) {
    return potts_buf_bytes(3 * n_member, count) + ((size_t)n_member * 2 + 15) / 16 * 16;
}

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

// Z3: work unit `gunit` = (instance, orbit); base[o] = first element of member o.  Member 0 is the tile whose
// HIGHEST outside digit is 0 (the orbit index enumerates the other outside digits, lowest first); member o
// adds o to every outside digit.  Consecutive orbits then differ in the lowest outside digit, so the units that
// run at the same time on neighbouring CTAs cover, member by member, rows that continue one another in memory
// (with the lowest digit fixed instead, neighbouring rows belong to far-away orbits: 3.3x read over-fetch).
struct PottsOrbit { unsigned inst, base[3]; };
__device__ __forceinline__ PottsOrbit potts_orbit(const PassParams& p, unsigned gunit) {
    const unsigned opi = (unsigned)(p.tiles_per_inst / 3);
    PottsOrbit t;
    t.inst = gunit / opi;
    unsigned rest = gunit - t.inst * opi;           // the top outside digit of member 0 is 0: it runs out of `rest`
    t.base[0] = t.base[1] = t.base[2] = 0u;
    auto take = [&](unsigned pw) {
        const unsigned d = rest % 3u; rest /= 3u;
        t.base[0] += d * pw; t.base[1] += ((d + 1u) % 3u) * pw; t.base[2] += ((d + 2u) % 3u) * pw;
    };
    unsigned pw = (unsigned)p.P_lo;
    for (int c = p.lo; c < p.a; ++c, pw *= 3u) take(pw);          // columns between the riding and the high block
    pw = (unsigned)p.P_b;
    for (int c = p.b; c < p.L; ++c, pw *= 3u) take(pw);           // columns above the tile
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
    const unsigned Nm = p.n_tile;                                           // elements per (member) tile
    const int NMEM = p.z3 ? 3 : 1;                                          // Z3: the three tiles of a rotation orbit
    const unsigned N = Nm * (unsigned)NMEM;
    double* sn = reinterpret_cast<double*>(smem_raw);                       // [N] if COUNT
    float* sx = reinterpret_cast<float*>(smem_raw + (COUNT ? (size_t)N * 8 : 0));
    unsigned short* s_rot = reinterpret_cast<unsigned short*>(smem_raw + potts_buf_bytes(N, COUNT));   // [Nm] (Z3)
    __shared__ int s_dig[3][GMAX_L + 1];     // per member: digits of the tile's base index; slot GMAX_L = 0 ("no such column")
    __shared__ float s_fin[GMAX_L];          // K_c of A_{L-1} (REDUCE pass)
    __shared__ float s_k00;                  // Z3: the bond column 0 - column 1 of A_{L-1}
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
    const unsigned m_nm = fastdiv_magic(Nm);
    const bool init = p.flags & PASS_INIT, reduce = p.flags & PASS_REDUCE;

    // per-gate index constants that do not depend on the tile
    for (int i = threadIdx.x; i < p.n_ops; i += THREADS) {
        const Op o = p.ops[i];
        if (o.pos == VCOL) { s_aux[i] = make_uint4(0u, 0u, 0u, 1u << 2); continue; }     // column-0 gate: no tile digit
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
    if (p.z3)                                 // r1: every local digit minus 1 (mod 3)
        for (unsigned e = threadIdx.x; e < Nm; e += THREADS) {
            unsigned rest = e, pw = 1, out = 0;
            for (int j = 0; j < p.T; ++j) { const unsigned d = rest % 3u; rest /= 3u; out += ((d + 2u) % 3u) * pw; pw *= 3u; }
            s_rot[e] = (unsigned short)out;
        }
    if (threadIdx.x == 0) {
        s_dig[0][GMAX_L] = s_dig[1][GMAX_L] = s_dig[2][GMAX_L] = 0;
        int nblk = 0;
        for (int i = 0; i < p.n_ops; ++i) if (p.ops[i].nb) s_list[nblk++] = (unsigned char)i;
        s_nblk = nblk;
    }

    unsigned last_inst = 0xffffffffu;
    for (unsigned gtile = blockIdx.x; gtile < total_tiles; gtile += gridDim.x) {
        PottsOrbit tl;
        if (p.z3) tl = potts_orbit(p, gtile);
        else { const PottsTile t1 = potts_tile(p, gtile); tl.inst = t1.inst; tl.base[0] = tl.base[1] = tl.base[2] = t1.base; }
        __syncthreads();                     // everyone is done with the previous tile
        // ---- load (or initialise to the semiring one) ----------------------------------------
        if (init) {
            for (unsigned e = threadIdx.x; e < N; e += THREADS) { sx[e] = 0.f; if (COUNT) sn[e] = 1.0; }
        } else {
            const float* gx = p.src_x + (unsigned long long)tl.inst * p.src_stride;
            const double* gn = COUNT ? p.src_n + (unsigned long long)tl.inst * p.src_stride : nullptr;
            for (unsigned e = threadIdx.x; e < N; e += THREADS) {
                const unsigned mem = NMEM == 1 ? 0u : (Nm == 1u ? e : fastdiv(e, m_nm)), le = e - mem * Nm;
                const unsigned row = plo == 1 ? le : fastdiv(le, m_plo);
                const unsigned off = tl.base[mem] + (le - row * plo) + row * pa;
                cp_async4(sx + e, gx + off);
                if (COUNT) cp_async8(sn + e, gn + off);
            }
        }
        for (int i = threadIdx.x; i < NMEM * p.L; i += THREADS) {   // digit c of the base index (0 for the tile's own columns)
            const int mem = i / p.L, cc = i - mem * p.L;
            unsigned pw = 1;
            for (int c = 0; c < cc; ++c) pw *= Q;
            s_dig[mem][cc] = (int)((tl.base[mem] / pw) % Q);
        }
        if (tl.inst != last_inst) {
            if (reduce) {
                for (int i = threadIdx.x; i < GMAX_L; i += THREADS) s_fin[i] = p.fin[(size_t)tl.inst * (2 * GMAX_L) + GMAX_L + i];
                if (threadIdx.x == 0) s_k00 = p.z3 ? p.fin[(size_t)tl.inst * (2 * GMAX_L)] : 0.f;
            }
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
            if (aux.x == 0u) {                                     // the gate on column 0 (Z3)
                potts_vgate<COUNT>(sx, sn, Nm, gk[0], s_rot, p.lo > 0 || p.a == 0, s_dig[0][0]);
            } else {
                const unsigned gpm = NMEM == 1 ? 0u : Nm / (nb == 3 ? 27u : (nb == 2 ? 9u : 3u));
                if (!COUNT && nb == 3) potts_block<3, COUNT>(sx, sn, N, aux, gk, s_dig, gpm);   // counting: blocks of <= 2
                else if (nb == 2) potts_block<2, COUNT>(sx, sn, N, aux, gk, s_dig, gpm);
                else potts_block<1, COUNT>(sx, sn, N, aux, gk, s_dig, gpm);
            }
            __syncthreads();
        }

        // ---- store, or multiply by A_{L-1}(s) and reduce ------------------------------------------
        if (reduce) {
            const float* K = s_fin;
            float bm_all = -INFINITY; double cnt_all = 0.0;          // (thread 0) over the members
            for (int mem = 0; mem < NMEM; ++mem) {
                const int* dig = s_dig[mem];
                float* mx_ = sx + (size_t)mem * Nm;
                const double* mn_ = sn + (size_t)mem * Nm;
                __syncthreads();
                if (threadIdx.x == 0) {              // bonds whose columns both lie outside the tile
                    float acc = 0.f;
                    for (int c = 0; c + 1 < p.L; ++c) {
                        const bool in_c = c < p.lo || (c >= p.a && c < p.b);
                        const bool in_n = c + 1 < p.lo || (c + 1 >= p.a && c + 1 < p.b);
                        if (!in_c && !in_n) acc += diag2<Q>(K[c], dig[c], dig[c + 1]);
                    }
                    if (p.z3 && p.lo == 0 && p.a > 0) acc += diag2<Q>(s_k00, 0, dig[0]);     // column 0 (colour 0) - digit 0 outside the tile
                    s_aout = acc;
                }
                __syncthreads();
                // A_{L-1}(s) restricted to the tile = table over the low (<= 4) tile digits + table over
                // the other (<= 5) digits + the one bond between the two groups
                const int GA = p.T < 4 ? p.T : 4;
                unsigned NA = 1;
                for (int i = 0; i < GA; ++i) NA *= Q;
                const unsigned NBH = Nm / NA, m_na = fastdiv_magic(NA);
                auto terms = [&](unsigned idx, int pos0, int pos1) {
                    float acc = 0.f;
                    unsigned rest = idx;
                    int dprev = 0, cprev = -2;
                    for (int pos = pos0; pos < pos1; ++pos) {
                        const int d = (int)(rest % Q); rest /= Q;
                        const int c = tile_col(p, pos);
                        if (c > 0) {
                            if (cprev == c - 1) acc += diag2<Q>(K[c - 1], dprev, d);                 // left neighbour in this group
                            else if (!(pos > 0 && tile_col(p, pos - 1) == c - 1)) acc += diag2<Q>(K[c - 1], dig[c - 1], d);   // outside the tile
                        }                                                                            // else: the bond between the groups
                        else if (p.z3) acc += diag2<Q>(s_k00, 0, d);                                 // digit 0 - column 0 (colour 0)
                        const bool right_in = pos + 1 < p.T && tile_col(p, pos + 1) == c + 1;
                        if (c + 1 < p.L && !right_in) acc += diag2<Q>(K[c], d, dig[c + 1]);
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
                for (unsigned e = threadIdx.x; e < Nm; e += THREADS) {
                    const unsigned hi = NA == Nm ? 0u : fastdiv(e, m_na), lo = e - hi * NA;
                    float acc = s_aout + s_tabA[lo] + s_tabB[hi];
                    if (lo / (NA / Q) == hi % Q) acc += Kx;
                    const float val = mx_[e] + acc;
                    mx_[e] = val;
                    mx = fmaxf(mx, val);
                }
                mx = warp_max(mx);
                if ((threadIdx.x & 31) == 0) red_x[threadIdx.x >> 5] = mx;
                __syncthreads();
                float bm = red_x[0];
                for (int w = 1; w < THREADS / 32; ++w) bm = fmaxf(bm, red_x[w]);
                double cnt = 0.0;
                if (COUNT) {
                    for (unsigned e = threadIdx.x; e < Nm; e += THREADS) if (mx_[e] == bm) cnt += mn_[e];
                    cnt = warp_sum(cnt);
                    if ((threadIdx.x & 31) == 0) red_n[threadIdx.x >> 5] = cnt;
                    __syncthreads();
                }
                if (threadIdx.x == 0) {
                    double tot = 0.0;
                    if (COUNT) for (int w = 0; w < THREADS / 32; ++w) tot += red_n[w];
                    if (bm > bm_all) { bm_all = bm; cnt_all = tot; } else if (bm == bm_all) cnt_all += tot;
                }
            }
            if (threadIdx.x == 0) {
                p.part_x[gtile] = bm_all;
                if (COUNT) p.part_n[gtile] = cnt_all;
            }
        } else {
            float* gx = p.dst_x + (unsigned long long)tl.inst * p.dst_stride;
            double* gn = COUNT ? p.dst_n + (unsigned long long)tl.inst * p.dst_stride : nullptr;
            for (unsigned e = threadIdx.x; e < N; e += THREADS) {
                const unsigned mem = NMEM == 1 ? 0u : (Nm == 1u ? e : fastdiv(e, m_nm)), le = e - mem * Nm;
                const unsigned row = plo == 1 ? le : fastdiv(le, m_plo);
                const unsigned off = tl.base[mem] + (le - row * plo) + row * pa;
                gx[off] = sx[e];
                if (COUNT) gn[off] = sn[e];
            }
        }
    }
}

}  // namespace ttn
