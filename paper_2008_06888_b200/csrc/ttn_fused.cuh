// ttn_fused.cuh -- fused register-phase pass kernel for the Ising Tropical<f32> sweep ("v4":
// diagonal frame + mirrored layouts; see planner.h for the frame, the layouts and the schedule).
//
// One launch = one HBM pass.  Each WARP owns a tile of 2^12 state elements,
// 128 per thread, and runs the pass's micro-op program on it with no CTA-level cooperation:
//   * conjugated max-plus gates (A2) PAPER.md:242 on a register digit:
//         a' = max(a, b + ka[n]),  b' = max(b, a + kb[n]),   n = the two neighbour bits of the index,
//     the row diagonals (A3), (A4) PAPER.md:247-252 folded into the 8 constants of the gate and
//     the common +Jv deferred to a scalar (ttn_api.cu): 1 FMNMX + 1/2 FADD2 per element.  One
//     set of 7 unrolled bodies (one per register bit) serves both layouts of a tile;
//   * layout exchanges A <-> B through the warp's private shared-memory region with 128-bit
//     (LOW) / 64-bit (HIGH) bank-conflict-free accesses, synchronised with __syncwarp only;
//   * the last pass adds the accumulated diagonal A_{L-1}(s) (a 128-entry table over the
//     register digits in 4 boundary variants + a per-thread scalar) and max-reduces.
// Global traffic: the LOW tile (columns 0..11) moves 128-byte lines straight between HBM and
// registers with immediate offsets; HIGH tiles (columns a..a+8 plus the riding columns 0..2 on
// the low lane bits) move whole 32-byte sectors, four per request, one mad.wide.u32 per address.
// The 4 warps of a HIGH group own the 4 sectors of every line and meet at a named barrier before
// they touch memory; where a tile spans few pages the NEXT tile is fetched with cp.async into the
// warp's own exchange region as soon as the last exchange of the current tile is done.
// The kernel is persistent (one CTA per SM, 12 warps); programs and gate constants are staged in
// shared memory once per launch and instance.  ELEM = 1 instantiates the same kernel for
// Tropical<i16> (two elements per 32-bit word, packed VIADDMNMX gates).
#pragma once
#include <cstdint>
#include <cuda_runtime.h>
#include "planner.h"

namespace ttn {

// Warps per CTA (one CTA per SM): 12 warps of <= 168 registers, 3 per scheduler.  For the HIGH
// kernel this needs the group barriers below: 12 free-running warps requesting scattered 32-byte
// sectors take 13-16 ms for a copy-only pass, synchronised 4-warp groups 9 ms.
#ifndef TTN_FWARPS_LOW
#define TTN_FWARPS_LOW 12
#endif
#ifndef TTN_FWARPS_HIGH
#define TTN_FWARPS_HIGH 12
#endif
// Tropical<i16>: 8 warps of <= 255 registers.  Measured at 32x32 (profiles/r01m.md): 12 / 8 / 4 warps
// = 220 / 202 / 210 ms; the gain is in the passes whose tiles span 512 pages (a = 23: 18.2 -> 15.9,
// 14.6 -> 11.5, 13.8 -> 9.7 ms) and in the LOW passes; f32 is fastest with 12 (336 / 359 / 387 ms).
#ifndef TTN_FWARPS_I16
#define TTN_FWARPS_I16 8
#endif
constexpr int FWARPS_LOW = TTN_FWARPS_LOW, FWARPS_HIGH = TTN_FWARPS_HIGH, FWARPS_I16 = TTN_FWARPS_I16;
constexpr int FREGION_F4 = 33 * 32;       // float4 per warp exchange region (low tile: padded rows)
constexpr int FMAX_MOPS = 128;            // micro-ops per pass
constexpr int FMAX_GATES = 160;           // gates per pass (8 constants each)
constexpr int FFINAL_FLOATS = 4 * 128 + 2 * 64;   // final table (4 variants) + H[64] + K[64]
__host__ __device__ constexpr int fwarps(bool low, int elem = 0) { return elem == 1 ? FWARPS_I16 : (low ? FWARPS_LOW : FWARPS_HIGH); }
__host__ __device__ constexpr size_t fsmem_bytes(bool low, int elem = 0) {
    return (size_t)fwarps(low, elem) * FREGION_F4 * 16 + (size_t)(FMAX_GATES + 1) * 32 + (size_t)FFINAL_FLOATS * 4 +
           (size_t)FMAX_MOPS * 4 + 64 + 256;       // + per-warp mbarriers and their phases (bulk prefetch)
}

struct FusedParams {
    int L, a, low, flags, first_layout, last_layout, batch;
    float* state;                       // instance 0: where the pass WRITES (and reads, unless src is set)
    unsigned long long inst_stride;     // elements between instances
    const float* src;                   // where the pass READS (row-aligned plans: a checkpoint); else = state
    unsigned long long src_stride;
    unsigned long long tiles_per_inst;  // warp tiles (2^12 elements) per instance
    const MicroOp* mops; int n_mops;    // this pass's program
    const float* gate_k; int n_gates;   // [inst][all gates][8]; this pass's slice of instance 0
    unsigned long long gate_inst_stride;          // floats between instances
    const float* final_tab;             // [inst][FFINAL_FLOATS] (REDUCE pass only)
    float* part_x;                      // [batch][part_stride] (REDUCE)
    int prefetch_pc;                    // HIGH: -1 = synchronous loads (tiles spanning > 256 pages of 2 MiB:
                                        // the burst of a whole tile's translations is slower than 128
                                        // paced loads); else the micro-op index after the last exchange: from
                                        // there on the warp's shared-memory region is free, and the NEXT
                                        // tile is fetched into it asynchronously (cp.async) while the rest
                                        // of this tile's gates run
    int cta_per_inst;                   // 1: few tiles per instance -- every CTA sweeps whole instances
    int igroup, tpi_shift;              // GROUP kernels: instances a CTA takes at a time (their tiles form one
                                        // flat list, so 16 tiles on 12 warps do not cost two full rounds each);
                                        // log2(tiles_per_inst)
                                        // (blockIdx.x, + gridDim.x, ...) with its own warps only
    int part_stride;                    // partials per instance: gridDim.x, or 1 when cta_per_inst
    int L_cols;                         // Tropical<i16> only: lattice L (p.L = L - 1 word digits)
    unsigned stride_bytes;              // HIGH: 4 << a, passed opaque so that the address math stays
                                        // one mad.wide.u32 (32 x 32 -> 64 bit) per access
    float* ckpt;                        // merged row plans: where MC_CKPT stores the tile (instance 0), else NULL
    unsigned long long ckpt_stride;
};

// (o0, o1) = (a0 + b0, a1 + b1) in one FADD2
__device__ __forceinline__ void add2(float& o0, float& o1, float a0, float a1, float b0, float b1) {
    asm("{ .reg .b64 ra, rb, rc;\n\t"
        "mov.b64 ra, {%2, %3};\n\t"
        "mov.b64 rb, {%4, %5};\n\t"
        "add.f32x2 rc, ra, rb;\n\t"
        "mov.b64 {%0, %1}, rc; }"
        : "=f"(o0), "=f"(o1) : "f"(a0), "f"(a1), "f"(b0), "f"(b1));
}

// FADD2 against a pre-packed 64-bit constant pair; unpacking of a 64-bit pair into two floats
__device__ __forceinline__ void add2p(float& o0, float& o1, float a0, float a1, unsigned long long kp) {
    asm("{ .reg .b64 ra, rc;\n\t"
        "mov.b64 ra, {%2, %3};\n\t"
        "add.f32x2 rc, ra, %4;\n\t"
        "mov.b64 {%0, %1}, rc; }"
        : "=f"(o0), "=f"(o1) : "f"(a0), "f"(a1), "l"(kp));
}
__device__ __forceinline__ void unpack2(unsigned long long p, float& lo, float& hi) {
    asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(p));
}

// ---- conjugated gate on register-index bit K ------------------------------------------------------
// PN / QN: register-index bit holding the P / Q neighbour (chain position -1 / +1), or -1 when
// that neighbour is constant per thread (its bit is then tp / tq).  a = the element whose bit K
// is 0.  The 8 constants ka[pn][qn], kb[pn][qn] arrive as two 128-bit shared-memory loads
// (c0, c1), stored by the prep kernel in the order this body wants (gate_order()):
//   ORDER_DEFAULT  c0 = ka[0][0] ka[0][1] ka[1][0] ka[1][1],  c1 = kb likewise
//   ORDER_K0       c0 = kb00 ka00 kb01 ka01,  c1 = kb10 ka10 kb11 ka11     (K = 0: pair = (a, b))
//   ORDER_PN0      c0 = ka[0][0] ka[1][0] ka[0][1] ka[1][1],  c1 = kb likewise   (bit 0 = P neighbour)
// so that whenever the two elements of a register pair (v[j], v[j+1]) take DIFFERENT constants,
// the constant pair is already an aligned 64-bit register pair straight out of the load (ptxas
// otherwise rebuilds it with two moves in front of every FADD2: +67 % instructions for K = 0).
enum GateOrder : int { ORDER_DEFAULT = 0, ORDER_K0 = 1, ORDER_PN0 = 2 };
__host__ __device__ constexpr int gate_order(int K, int PN) { return K == 0 ? ORDER_K0 : (PN == 0 ? ORDER_PN0 : ORDER_DEFAULT); }

template <int K, int PN, int QN>
__device__ __forceinline__ void cgate(float (&v)[128], const ulonglong2 c0, const ulonglong2 c1, const int tp, const int tq) {
    constexpr int B = 1 << K;
#define TTN_NP(j) (PN < 0 ? 0 : (((j) >> (PN < 0 ? 0 : PN)) & 1))
#define TTN_NQ(j) (QN < 0 ? 0 : (((j) >> (QN < 0 ? 0 : QN)) & 1))
    if (K == 0) {
        // pair (v[j], v[j+1]) = (a, b): t0 = a + kb (candidate for b), t1 = b + ka (candidate for a)
        static_assert(K != 0 || (PN >= 0 && QN >= 0), "bit 0 sits inside the chain");
        const unsigned long long kp[2][2] = {{c0.x, c0.y}, {c1.x, c1.y}};
#pragma unroll
        for (int j = 0; j < 128; j += 2) {
            float t0, t1;
            add2p(t0, t1, v[j], v[j + 1], kp[TTN_NP(j)][TTN_NQ(j)]);
            v[j] = fmaxf(v[j], t1);
            v[j + 1] = fmaxf(v[j + 1], t0);
        }
    } else if (PN == 0 || QN == 0) {
        // bit 0 is a neighbour: (v[j], v[j+1]) take the constants for that neighbour bit = 0 / 1;
        // the pair index is the OTHER neighbour's bit (a register bit, or tq when it is per thread)
        unsigned long long pa[2] = {c0.x, c0.y}, pb[2] = {c1.x, c1.y};
        constexpr int ON = PN == 0 ? QN : PN;          // the other neighbour
        if (ON < 0) { const int t = PN == 0 ? tq : tp; pa[0] = t ? pa[1] : pa[0]; pb[0] = t ? pb[1] : pb[0]; }
#define TTN_NO(j) (ON < 0 ? 0 : (((j) >> (ON < 0 ? 0 : ON)) & 1))
#pragma unroll
        for (int j = 0; j < 128; j += 2) {
            if ((j & B) == 0) {
                float a0, a1, b0, b1;
                add2p(a0, a1, v[j], v[j + 1], pb[TTN_NO(j)]);
                add2p(b0, b1, v[j + B], v[j + B + 1], pa[TTN_NO(j)]);
                v[j] = fmaxf(v[j], b0); v[j + 1] = fmaxf(v[j + 1], b1);
                v[j + B] = fmaxf(v[j + B], a0); v[j + B + 1] = fmaxf(v[j + B + 1], a1);
            }
        }
#undef TTN_NO
    } else {
        float ka[2][2], kb[2][2];
        unpack2(c0.x, ka[0][0], ka[0][1]); unpack2(c0.y, ka[1][0], ka[1][1]);
        unpack2(c1.x, kb[0][0], kb[0][1]); unpack2(c1.y, kb[1][0], kb[1][1]);
        if (PN < 0) {
#pragma unroll
            for (int h = 0; h < 2; ++h) { ka[0][h] = tp ? ka[1][h] : ka[0][h]; kb[0][h] = tp ? kb[1][h] : kb[0][h]; }
        }
        if (QN < 0) {
#pragma unroll
            for (int l = 0; l < 2; ++l) { ka[l][0] = tq ? ka[l][1] : ka[l][0]; kb[l][0] = tq ? kb[l][1] : kb[l][0]; }
        }
#pragma unroll
        for (int j = 0; j < 128; j += 2) {
            if ((j & B) == 0) {
                float a0, a1, b0, b1;
                add2(a0, a1, v[j], v[j + 1], kb[TTN_NP(j)][TTN_NQ(j)], kb[TTN_NP(j)][TTN_NQ(j)]);
                add2(b0, b1, v[j + B], v[j + B + 1], ka[TTN_NP(j)][TTN_NQ(j)], ka[TTN_NP(j)][TTN_NQ(j)]);
                v[j] = fmaxf(v[j], b0); v[j + 1] = fmaxf(v[j + 1], b1);
                v[j + B] = fmaxf(v[j + B], a0); v[j + B + 1] = fmaxf(v[j + B + 1], a1);
            }
        }
    }
#undef TTN_NP
#undef TTN_NQ
}

// register bit of the P / Q neighbour of the chain position held by register bit K (-1: per thread)
template <bool LOW, int K> struct Nbr {
    static constexpr int pos = fused_chain_pos(LOW, K);
    static constexpr int PN = pos == 0 ? -1 : fused_bit_of_digit(LOW, 0, pos - 1);
    static constexpr int QN = pos == F_RB - 1 ? -1 : fused_bit_of_digit(LOW, 0, pos + 1);
};

// One round: for every set bit of `mask` (ascending) the next gate of that register digit.  The
// constants of the gate after the current one are already in flight (n0, n1): the gate list of a
// pass is contiguous in execution order, so the prefetch simply runs one entry ahead.
template <bool LOW>
__device__ __forceinline__ void fround(float (&v)[128], const unsigned mask, const ulonglong2* __restrict__& gk,
                                       ulonglong2& n0, ulonglong2& n1, const int tp, const int tq) {
#define TTN_FETCHK const ulonglong2 c0 = n0, c1 = n1; gk += 2; n0 = gk[0]; n1 = gk[1];
#define TTN_G(Kk)                                                                                   \
    if (mask & (1u << Kk)) {                                                                        \
        TTN_FETCHK                                                                                  \
        cgate<Kk, Nbr<LOW, Kk>::PN, Nbr<LOW, Kk>::QN>(v, c0, c1, tp, tq);                           \
    }
    TTN_G(0) TTN_G(1) TTN_G(2) TTN_G(3) TTN_G(4) TTN_G(5) TTN_G(6)
#undef TTN_G
}

// ---- Z2 flip gate (h = 0; planner.h "GLOBAL-FLIP (Z2) REDUCTION") -------------------------------------
// The stored half-state obeys W[s_0 = 1, u] = W[s_0 = 0, ~u], so the gate (A2) on column 0 reads
//     W'[u] = max(W[u], W[~u] + kf[bit of column 1 in u]).
// ~u lives in the complement tile, which the partner warp (warp ^ 1) of the pair holds in the same
// layout: both warps publish their registers in their own exchange region (the store half of an
// exchange), meet at the pair's named barrier, and read the partner's region at the complemented
// position -- register 127 - j of lane 31 - lane -- which mirrors the load half of the exchange and
// is bank-conflict free for the same reason.  A second barrier frees the regions.
__device__ __forceinline__ void pair_sync(int warp) {
    asm volatile("bar.sync %0, 64;" :: "r"(1 + (warp >> 1)) : "memory");
}
__host__ __device__ constexpr int rev5c(int q) {
    return ((q & 1) << 4) | ((q & 2) << 2) | (q & 4) | ((q & 8) >> 2) | ((q & 16) >> 4);
}
template <int LAYOUT>
__device__ __forceinline__ void flipgate(float (&v)[128], float4* myreg, const float4* preg, const int lane,
                                         const int warp, const float k0, const float k1) {
    __syncwarp();
    if (LAYOUT == 0) {
        float4* p = myreg + 33 * lane;
#pragma unroll
        for (int q = 0; q < 32; ++q) p[q] = make_float4(v[4 * q], v[4 * q + 1], v[4 * q + 2], v[4 * q + 3]);
    } else {
        float4* p = myreg + lane;
#pragma unroll
        for (int q = 0; q < 32; ++q) p[33 * rev5c(q)] = make_float4(v[4 * q], v[4 * q + 2], v[4 * q + 1], v[4 * q + 3]);
    }
    pair_sync(warp);
    if (LAYOUT == 0) {          // column 1 = tile digit 0 = register bit 2 = bit 0 of the quad index
        const float4* p = preg + 33 * (31 - lane);
#pragma unroll
        for (int q = 0; q < 32; ++q) {
            const float4 t = p[31 - q];
            const float kq = (q & 1) ? k1 : k0;
            float a0, a1, a2, a3;
            add2(a0, a1, t.w, t.z, kq, kq);
            add2(a2, a3, t.y, t.x, kq, kq);
            v[4 * q] = fmaxf(v[4 * q], a0); v[4 * q + 1] = fmaxf(v[4 * q + 1], a1);
            v[4 * q + 2] = fmaxf(v[4 * q + 2], a2); v[4 * q + 3] = fmaxf(v[4 * q + 3], a3);
        }
    } else {                    // column 1 = lane bit 0
        const float4* p = preg + (31 - lane);
        const float kk = (lane & 1) ? k1 : k0;
#pragma unroll
        for (int q = 0; q < 32; ++q) {
            const float4 t = p[33 * rev5c(31 - q)];
            float a0, a1, a2, a3;
            add2(a0, a1, t.w, t.y, kk, kk);
            add2(a2, a3, t.z, t.x, kk, kk);
            v[4 * q] = fmaxf(v[4 * q], a0); v[4 * q + 1] = fmaxf(v[4 * q + 1], a1);
            v[4 * q + 2] = fmaxf(v[4 * q + 2], a2); v[4 * q + 3] = fmaxf(v[4 * q + 3], a3);
        }
    }
    pair_sync(warp);
}

// Tropical<i16> form: column 1 is the half of a word, so ~u = the OTHER half of the complement word,
// and the neighbour bit of the flip gate is the half itself: one PRMT + one VIADDMNMX.S16x2 per word
// against the packed constant kpk = (lo: kf[0], hi: kf[1]).
template <int LAYOUT>
__device__ __forceinline__ void flipgate16(float (&v)[128], float4* myreg, const float4* preg, const int lane,
                                           const int warp, const unsigned kpk) {
    __syncwarp();
    if (LAYOUT == 0) {
        float4* p = myreg + 33 * lane;
#pragma unroll
        for (int q = 0; q < 32; ++q) p[q] = make_float4(v[4 * q], v[4 * q + 1], v[4 * q + 2], v[4 * q + 3]);
    } else {
        float4* p = myreg + lane;
#pragma unroll
        for (int q = 0; q < 32; ++q) p[33 * rev5c(q)] = make_float4(v[4 * q], v[4 * q + 2], v[4 * q + 1], v[4 * q + 3]);
    }
    pair_sync(warp);
    auto upd = [&](float& x, float pw) {
        const unsigned sw = __byte_perm(__float_as_uint(pw), 0u, 0x1032);       // the partner's other half
        x = __uint_as_float(__viaddmax_s16x2(sw, kpk, __float_as_uint(x)));
    };
    if (LAYOUT == 0) {
        const float4* p = preg + 33 * (31 - lane);
#pragma unroll
        for (int q = 0; q < 32; ++q) {
            const float4 t = p[31 - q];
            upd(v[4 * q], t.w); upd(v[4 * q + 1], t.z); upd(v[4 * q + 2], t.y); upd(v[4 * q + 3], t.x);
        }
    } else {
        const float4* p = preg + (31 - lane);
#pragma unroll
        for (int q = 0; q < 32; ++q) {
            const float4 t = p[33 * rev5c(31 - q)];
            upd(v[4 * q], t.w); upd(v[4 * q + 1], t.y); upd(v[4 * q + 2], t.z); upd(v[4 * q + 3], t.x);
        }
    }
    pair_sync(warp);
}

// ---- Tropical<i16> (the paper's own Int16 choice for +-J) -----------
// Two elements per 32-bit word: column 0 of the lattice row is the HALF of a word (low half =
// bit 0 = sigma +1), the kernel's tile geometry applies to the word index.  One VIADDMNMX.S16x2
// does max(b + k, a) for both halves: 1 alu-pipe instruction per word and gate, no fma-pipe add.
// Constants are packed per half (lo = element with column-0 bit 0) by the prep kernel.
__device__ __forceinline__ float vam2(float b, unsigned k, float a) {
    return __uint_as_float(__viaddmax_s16x2(__float_as_uint(b), k, __float_as_uint(a)));
}
template <int K, int PN, int QN>
__device__ __forceinline__ void cgate16(float (&v)[128], const uint4 c0, const uint4 c1, const int tp, const int tq) {
    unsigned ka[2][2] = {{c0.x, c0.y}, {c0.z, c0.w}}, kb[2][2] = {{c1.x, c1.y}, {c1.z, c1.w}};
    if (PN < 0) {
#pragma unroll
        for (int h = 0; h < 2; ++h) { ka[0][h] = tp ? ka[1][h] : ka[0][h]; kb[0][h] = tp ? kb[1][h] : kb[0][h]; }
    }
    if (QN < 0) {
#pragma unroll
        for (int l = 0; l < 2; ++l) { ka[l][0] = tq ? ka[l][1] : ka[l][0]; kb[l][0] = tq ? kb[l][1] : kb[l][0]; }
    }
    constexpr int B = 1 << K;
#pragma unroll
    for (int j = 0; j < 128; ++j) {
        if (j & B) continue;
        const int np = PN < 0 ? 0 : (j >> (PN < 0 ? 0 : PN)) & 1, nq = QN < 0 ? 0 : (j >> (QN < 0 ? 0 : QN)) & 1;
        const float a = v[j], b = v[j + B];
        v[j] = vam2(b, ka[np][nq], a);
        v[j + B] = vam2(a, kb[np][nq], b);
    }
}
// gate on column 0 (the half of a word): partner = the other half of the same word.  kp[n] =
// (lo: ka, hi: kb) for column-1 bit n; Q1 = register bit holding column 1, or -1 (then t1).
template <int Q1>
__device__ __forceinline__ void hgate16(float (&v)[128], const uint4 c0, const int t1) {
    unsigned kp[2] = {c0.x, c0.y};
    if (Q1 < 0) kp[0] = t1 ? kp[1] : kp[0];
#pragma unroll
    for (int j = 0; j < 128; ++j) {
        const unsigned w = __float_as_uint(v[j]);
        const unsigned sw = __byte_perm(w, 0u, 0x1032);           // swap the halves
        v[j] = __uint_as_float(__viaddmax_s16x2(sw, kp[Q1 < 0 ? 0 : (j >> (Q1 < 0 ? 0 : Q1)) & 1], w));
    }
}
template <bool LOW>
__device__ __forceinline__ void fround16(float (&v)[128], const unsigned mask, const uint4* __restrict__ gk,
                                         const int layout, const int tp, const int tq, const int t1) {
#define TTN_G16(Kk)                                                                                 \
    if (mask & (1u << Kk)) {                                                                        \
        const uint4 c0 = gk[0], c1 = gk[1]; gk += 2;                                                \
        cgate16<Kk, Nbr<LOW, Kk>::PN, Nbr<LOW, Kk>::QN>(v, c0, c1, tp, tq);                         \
    }
    TTN_G16(0) TTN_G16(1) TTN_G16(2) TTN_G16(3) TTN_G16(4) TTN_G16(5) TTN_G16(6)
#undef TTN_G16
    if (LOW && (mask & 0x80u)) {             // column 0; column 1 = tile digit 0 = register bit 2 in layout A, lane bit 0 in B
        const uint4 c0 = gk[0];
        if (layout == 0) hgate16<fused_bit_of_digit(true, 0, 0)>(v, c0, 0); else hgate16<-1>(v, c0, t1);
    }
}

// ---- layout exchange through the warp's shared-memory region ----------------------------------------
// LOW (128-bit): a float4 holds the 4 elements differing in (d5, d6), in layout A's register
//   order (.x: d5=0,d6=0  .y: d5=1  .z: d6=1  .w: both); float4 index = (d0..d4) + 33 (d7..d11).
//     A (lanes d7..d11, quad bits = d0..d4): 33 lane + q
//     B (lanes d0..d4, quad bits = d11..d7, register bits 0,1 = d6,d5): lane + 33 rev5(q), and
//       the two middle elements of the quad swap places.
// HIGH (64-bit): a float2 holds the 2 elements differing in d4 (register bit 0 in both layouts);
//   float2 index = rho + 8 (d0^d7) + 16 d7 + 32 d1 + 64 d2 + 128 d3 + 256 d5 + 512 d6 + 1024 d8
//   (the XOR puts a lane digit of either layout on bank bit 3: conflict-free half-warps).
//     A (lanes rho,d7,d8; pair bits = d5,d6,d0,d1,d2,d3)   B (lanes rho,d0,d1; pair bits = d3,d2,d8,d7,d6,d5)
__host__ __device__ constexpr int rev5(int q) {
    return ((q & 1) << 4) | ((q & 2) << 2) | (q & 4) | ((q & 8) >> 2) | ((q & 16) >> 4);
}
__host__ __device__ constexpr int xh_imm_a(int pr) {   // pr = j >> 1: bits d5,d6,d0,d1,d2,d3 ; d0 goes to the base
    return 256 * (pr & 1) + 512 * ((pr >> 1) & 1) + 32 * ((pr >> 3) & 1) + 64 * ((pr >> 4) & 1) + 128 * ((pr >> 5) & 1);
}
__host__ __device__ constexpr int xh_imm_b(int pr) {   // pr bits d3,d2,d8,d7,d6,d5 ; d7 goes to the base
    return 128 * (pr & 1) + 64 * ((pr >> 1) & 1) + 1024 * ((pr >> 2) & 1) + 512 * ((pr >> 4) & 1) + 256 * ((pr >> 5) & 1);
}

template <bool LOW, int LAYOUT, bool STORE>
__device__ __forceinline__ void xmove(float (&v)[128], float4* reg, int lane) {
    if (LOW) {
        if (LAYOUT == 0) {
            float4* p = reg + 33 * lane;
#pragma unroll
            for (int q = 0; q < 32; ++q) {
                if (STORE) p[q] = make_float4(v[4 * q], v[4 * q + 1], v[4 * q + 2], v[4 * q + 3]);
                else { const float4 t = p[q]; v[4 * q] = t.x; v[4 * q + 1] = t.y; v[4 * q + 2] = t.z; v[4 * q + 3] = t.w; }
            }
        } else {
            float4* p = reg + lane;
#pragma unroll
            for (int q = 0; q < 32; ++q) {
                if (STORE) p[33 * rev5(q)] = make_float4(v[4 * q], v[4 * q + 2], v[4 * q + 1], v[4 * q + 3]);
                else { const float4 t = p[33 * rev5(q)]; v[4 * q] = t.x; v[4 * q + 1] = t.z; v[4 * q + 2] = t.y; v[4 * q + 3] = t.w; }
            }
        }
    } else {
        float2* r2 = reinterpret_cast<float2*>(reg);
        const int rho = lane & 7, l3 = (lane >> 3) & 1, l4 = (lane >> 4) & 1;
        if (LAYOUT == 0) {          // l3 = d7, l4 = d8; base per d0 (pair bit 2)
            float2* b0 = r2 + rho + 8 * l3 + 16 * l3 + 1024 * l4;
            float2* b1 = r2 + rho + 8 * (1 - l3) + 16 * l3 + 1024 * l4;
#pragma unroll
            for (int pr = 0; pr < 64; ++pr) {
                float2* p = (((pr >> 2) & 1) ? b1 : b0) + xh_imm_a(pr);
                if (STORE) *p = make_float2(v[2 * pr], v[2 * pr + 1]);
                else { const float2 t = *p; v[2 * pr] = t.x; v[2 * pr + 1] = t.y; }
            }
        } else {                    // l3 = d0, l4 = d1; base per d7 (pair bit 3)
            float2* b0 = r2 + rho + 8 * l3 + 32 * l4;
            float2* b1 = r2 + rho + 8 * (1 - l3) + 16 + 32 * l4;
#pragma unroll
            for (int pr = 0; pr < 64; ++pr) {
                float2* p = (((pr >> 3) & 1) ? b1 : b0) + xh_imm_b(pr);
                if (STORE) *p = make_float2(v[2 * pr], v[2 * pr + 1]);
                else { const float2 t = *p; v[2 * pr] = t.x; v[2 * pr + 1] = t.y; }
            }
        }
    }
}

// ---- global <-> register: element index e (inside the warp tile) of register j ---------------
//   LOW  B: e = lane + 32 (d5 + 2 d6 + ... + 64 d11), register bits = d6,d5,d11,d10,d9,d8,d7
//   HIGH A: e = 16 b0 + 32 b1 + 64 b2 + b3 + 2 b4 + 4 b5 + 8 b6 + 128 (lane >> 3)
//   HIGH B: e = 16 b0 +  8 b1 +  4 b2 + 256 b3 + 128 b4 + 64 b5 + 32 b6 + (lane >> 3)
//   (address = tile base + rho + (e << a) for HIGH)
__host__ __device__ constexpr int ereg_low_b(int j) {
    return 2 * (j & 1) + ((j >> 1) & 1) + 64 * ((j >> 2) & 1) + 32 * ((j >> 3) & 1) + 16 * ((j >> 4) & 1) +
           8 * ((j >> 5) & 1) + 4 * ((j >> 6) & 1);
}
__host__ __device__ constexpr int ereg_high(int layout, int j) {
    return layout == 0
        ? 16 * (j & 1) + 32 * ((j >> 1) & 1) + 64 * ((j >> 2) & 1) + ((j >> 3) & 1) + 2 * ((j >> 4) & 1) +
          4 * ((j >> 5) & 1) + 8 * ((j >> 6) & 1)
        : 16 * (j & 1) + 8 * ((j >> 1) & 1) + 4 * ((j >> 2) & 1) + 256 * ((j >> 3) & 1) + 128 * ((j >> 4) & 1) +
          64 * ((j >> 5) & 1) + 32 * ((j >> 6) & 1);
}

// address of element offset (imm * stride) from a 64-bit base: mad.wide.u32; `sb` is the stride
// in bytes as an opaque 32-bit value.  ptxas 12.9 lowers it to IMAD.WIDE.U32 (product, fma pipe) +
// IADD3 + IMAD.X (64-bit add).  The C++ spelling `gbase + (u64)sb * imm` does become ONE
// IMAD.WIDE.U32 with a 64-bit addend (the HIGH kernel shrinks from 5096 to 4072 SASS instructions)
// but the sweep is SLOWER with it (32x32: 338.8 vs 336.6 ms, profiles/r01m.md), so this form stays.
// The result is a GLOBAL-space address: the accesses below are spelled ld.global / st.global
// because a pointer that comes out of inline asm is "generic" to the compiler (LD/ST instead of
// LDG/STG).
__device__ __forceinline__ unsigned long long addr_mad(unsigned long long gbase, unsigned sb, unsigned imm) {
    unsigned long long r;
    asm("mad.wide.u32 %0, %1, %2, %3;" : "=l"(r) : "r"(sb), "r"(imm), "l"(gbase));
    return r;
}
__device__ __forceinline__ float ldg_f32(unsigned long long ga) {
    float x;
    asm volatile("ld.global.f32 %0, [%1];" : "=f"(x) : "l"(ga));
    return x;
}
__device__ __forceinline__ void stg_f32(unsigned long long ga, float x) {
    asm volatile("st.global.f32 [%0], %1;" :: "l"(ga), "f"(x) : "memory");
}

template <bool LOW, int LAYOUT, bool STORE>
__device__ __forceinline__ void gmove(float (&v)[128], float* tile, int lane, unsigned sb, int a) {
    if (LOW) {
        float* p = tile + lane;                                   // layout B only (planner guarantees)
#pragma unroll
        for (int j = 0; j < 128; ++j) { if (STORE) p[32 * ereg_low_b(j)] = v[j]; else v[j] = p[32 * ereg_low_b(j)]; }
        return;
    }
    // HIGH: element e of the tile sits at tile + rho + (e << a); per-lane part first
    const unsigned elane = (LAYOUT == 0) ? 128u * (unsigned)(lane >> 3) : (unsigned)(lane >> 3);
    const unsigned long long p = (unsigned long long)__cvta_generic_to_global(tile + (lane & 7) + ((unsigned long long)elane << a));
#pragma unroll
    for (int j = 0; j < 128; ++j) {      // 32 x 32 -> 64-bit product: valid for sb < 2^32 (a <= 29)
        const unsigned long long q = addr_mad(p, sb, (unsigned)ereg_high(LAYOUT, j));
        if (STORE) stg_f32(q, v[j]); else v[j] = ldg_f32(q);
    }
}

// ---- last pass: v[j] += A_{L-1}(s) -------------------------------------------------------------------
// s_fin = [4 variants][128] table over the register digits (variant = tl + 2 th: the boundary
// couplings to the columns left / right of the 7 register columns) followed by H[64], K[64]
// (accumulated fields and horizontal couplings).  x0 = first register column; sthr = the
// element index with the register digits cleared.
__device__ __forceinline__ float final_thread_const(const float* s_fin, int L, int x0, unsigned long long sthr) {
    const float* H = s_fin + 512; const float* Kc = s_fin + 576;
    float acc = 0.f;
    for (int c = 0; c < L; ++c) {
        const bool in_r = (c >= x0 && c < x0 + F_RB);
        const int bc = (int)((sthr >> c) & 1ull);
        if (!in_r) acc += bc ? -H[c] : H[c];
        if (c + 1 < L) {
            const bool in_r1 = (c + 1 >= x0 && c + 1 < x0 + F_RB);
            if (!in_r && !in_r1) {
                const int b1 = (int)((sthr >> (c + 1)) & 1ull);
                acc += (bc == b1) ? Kc[c] : -Kc[c];
            }
        }
    }
    return acc;
}

// ---- HIGH tiles: asynchronous prefetch of the next tile into the warp's own exchange region -------
// Layout in the region: row e (512 rows of 8 floats = one 32-byte sector each) at float index
// 8 (e + (e >> 7)): one slot of skew per 128 rows makes the reads of BOTH layouts bank-conflict
// free (layout A lanes differ in e by multiples of 128, layout B lanes by 1, 2, 3).
__device__ __forceinline__ void pf_issue(float4* region, const float* tile, int lane, unsigned sb, int a) {
    const unsigned sbase = (unsigned)__cvta_generic_to_shared(region) + 32u * (unsigned)(lane >> 1) + 16u * (unsigned)(lane & 1);
    const unsigned long long g = (unsigned long long)__cvta_generic_to_global(tile + ((unsigned long long)(lane >> 1) << a) + 4 * (lane & 1));
#pragma unroll
    for (int i = 0; i < 32; ++i) {       // rows e = 16 i + (lane >> 1), half h = lane & 1
        const unsigned long long ga = addr_mad(g, sb, 16u * i);
        asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" :: "r"(sbase + 32u * (16u * i + (i >> 3))), "l"(ga) : "memory");
    }
    asm volatile("cp.async.commit_group;" ::: "memory");
}
template <int LAYOUT>
__device__ __forceinline__ void pf_read(float (&v)[128], const float4* region, int lane) {
    const float* r = reinterpret_cast<const float*>(region);
    if (LAYOUT == 1) {                   // lanes (rho, d0, d1): e = (lane >> 3) + ereg, no carry into bit 7
        const float* q = r + lane;
#pragma unroll
        for (int j = 0; j < 128; ++j) v[j] = q[8 * (ereg_high(1, j) + (ereg_high(1, j) >> 7))];
    } else {                             // lanes (rho, d7, d8): e = ereg + 128 k, k = lane >> 3
        const float* q = r + (lane & 7) + 1032 * (lane >> 3);
#pragma unroll
        for (int j = 0; j < 128; ++j) v[j] = q[8 * ereg_high(0, j)];
    }
}

// LOW tiles: a contiguous 16 KiB tile is ONE bulk copy of the TMA unit (cp.async.bulk global -> shared,
// UBLKCP in SASS) issued by lane 0 and tracked by the warp's own mbarrier: no per-lane address arithmetic,
// no LSU instructions.  The region holds the tile linearly, read back in layout B (lanes = the 5 lowest
// digits).  The region was last touched by generic-proxy accesses (an exchange): fence.proxy.async
// orders them before the async-proxy write.
__device__ __forceinline__ void mbar_init(unsigned long long* mbar) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" :: "r"((unsigned)__cvta_generic_to_shared(mbar)) : "memory");
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void pf_issue_low(float4* region, const float* tile, int lane, unsigned long long* mbar) {
    __syncwarp();
    if (lane == 0) {
        const unsigned dst = (unsigned)__cvta_generic_to_shared(region), mb = (unsigned)__cvta_generic_to_shared(mbar);
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], 16384;" :: "r"(mb) : "memory");
        asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], 16384, [%2];"
                     :: "r"(dst), "l"((unsigned long long)__cvta_generic_to_global(tile)), "r"(mb) : "memory");
    }
}
__device__ __forceinline__ void pf_wait_low(unsigned long long* mbar, unsigned& phase) {
    const unsigned mb = (unsigned)__cvta_generic_to_shared(mbar);
    unsigned ok;
    do {
        asm volatile("{ .reg .pred p;\n\t"
                     "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
                     "selp.u32 %0, 1, 0, p; }" : "=r"(ok) : "r"(mb), "r"(phase) : "memory");
    } while (!ok);
    phase ^= 1u;
}
__device__ __forceinline__ void pf_read_low(float (&v)[128], const float4* region, int lane) {
    const float* q = reinterpret_cast<const float*>(region) + lane;
#pragma unroll
    for (int j = 0; j < 128; ++j) v[j] = q[32 * ereg_low_b(j)];
}

// named barrier of one 4-warp group (barrier 0 is __syncthreads)
__device__ __forceinline__ void group_sync(int warp) {
    asm volatile("bar.sync %0, 128;" :: "r"(1 + (warp >> 2)) : "memory");
}

// ELEM = 0: Tropical<f32>.  ELEM = 1: Tropical<i16>, two elements per word; then p.L, p.a and the
// tile geometry count WORD digits (column c >= 1 = word digit c - 1) and p.L_cols = lattice L.
// GROUP (cta_per_inst passes without a reduction, f32): a CTA stages the constants of p.igroup
// instances and walks their tiles as one list.
// One fused pass.  The body lives in ttn_fused_body.inc (see there).
template <bool LOW, int ELEM, bool GROUP>
__device__ __forceinline__ void fused_pass_body(const FusedParams& p, unsigned char* fsm_raw,
                                                const int inst_first, const int inst_step) {
    constexpr bool RED = false;          // GROUP passes never reduce
    constexpr bool Z2 = false;
    constexpr bool INIT_MBAR = false;    // fused_sweep_kernel initialises the mbarriers once
#include "ttn_fused_body.inc"
}

// RED = the last pass of a sweep (adds A_{L-1}(s) and reduces instead of storing)
// Z2 (LOW only) = the flip-reduced state: warps work in pairs on tiles (T, ~T) and the program may
// contain flip gates (planner.h "GLOBAL-FLIP (Z2) REDUCTION")
template <bool LOW, int ELEM = 0, bool GROUP = false, bool RED = false, bool Z2 = false>
__global__ void __launch_bounds__(fwarps(LOW, ELEM) * 32, 1) fused_pass_kernel(const FusedParams p) {
    extern __shared__ __align__(16) unsigned char fsm_raw[];
    const int inst_first = p.cta_per_inst ? (int)blockIdx.x * (GROUP ? p.igroup : 1) : 0;
    const int inst_step = p.cta_per_inst ? (int)gridDim.x * (GROUP ? p.igroup : 1) : 1;
    constexpr bool INIT_MBAR = true;
#include "ttn_fused_body.inc"
}

// Batches of small lattices (every pass in cta_per_inst mode, no reduction pass -- the row-aligned
// plans of ttn_ground_config): the instances are independent, so ONE launch runs all passes; a
// CTA takes p.igroup instances through the whole list of passes (block barrier between passes:
// the tiles of a pass are written by other warps of the same CTA) before it moves to its next
// instances.  Saves the launch gap and the ramp / tail of ~30 short kernels.
template <int ELEM = 0>
__global__ void __launch_bounds__(fwarps(true) * 32, 1) fused_sweep_kernel(const FusedParams* __restrict__ passes,
                                                                            const int n_passes) {
    static_assert(fwarps(true) == fwarps(false), "one CTA shape for both tile kinds");
    extern __shared__ __align__(16) unsigned char fsm_raw[];
    __shared__ FusedParams s_p;
    const int igroup = passes[0].igroup, batch = passes[0].batch;
    {   // the warps' mbarriers (bulk prefetch of LOW tiles) and their phases live behind s_red (ttn_fused_body.inc)
        unsigned long long* mb = reinterpret_cast<unsigned long long*>(fsm_raw + fsmem_bytes(true) - 256);
        if ((threadIdx.x & 31) == 0) { mbar_init(mb + (threadIdx.x >> 5)); reinterpret_cast<unsigned*>(mb + 16)[threadIdx.x >> 5] = 0u; }
        __syncthreads();
    }
    for (int inst = (int)blockIdx.x * igroup; inst < batch; inst += (int)gridDim.x * igroup) {
        for (int k = 0; k < n_passes; ++k) {
            __syncthreads();                                   // the previous pass is complete (and s_p free)
            for (int i = threadIdx.x; i < (int)(sizeof(FusedParams) / 4); i += blockDim.x)
                reinterpret_cast<unsigned*>(&s_p)[i] = reinterpret_cast<const unsigned*>(passes + k)[i];
            __syncthreads();
            if (s_p.low) fused_pass_body<true, ELEM, true>(s_p, fsm_raw, inst, 1 << 30);
            else fused_pass_body<false, ELEM, true>(s_p, fsm_raw, inst, 1 << 30);
        }
    }
}

// ---- S0: per-instance gate constants and the final table from the couplings ------------------------
struct FusedPrepParams {
    int L, n_gates;
    const int* gate_rc;            // [n_gates]  low << 16 | K << 13 | layout << 12 | r << 6 | c
    const float* Jh; const float* Jv; const float* h;   // device couplings, per instance
    float* gate_k;                 // [inst][n_gates][8]
    float* final_tab;              // [inst][FFINAL_FLOATS]
    int fin_low, fin_layout, fin_a;   // tile kind, layout and start column of the last pass's end
    int col_off;                   // Z2: 1 = the kernel's digit d is lattice column d + 1 (fin_a is a digit)
};

__global__ void __launch_bounds__(256) fused_prep_kernel(const FusedPrepParams p) {
    const unsigned long long inst = blockIdx.y;
    const int L = p.L;
    const float* Jh = p.Jh + inst * (unsigned long long)(L * (L - 1));
    const float* Jv = p.Jv + inst * (unsigned long long)((L - 1) * L);
    const float* hh = p.h ? p.h + inst * (unsigned long long)(L * L) : nullptr;
    const long idx = (long)blockIdx.x * blockDim.x + threadIdx.x;
    // accumulated diagonal coefficients through row R-1 (A_{R-1}), in double
    auto Hacc = [&](int R, int c) { double s = 0; if (hh) for (int r = 0; r < R; ++r) s += (double)hh[r * L + c]; return s; };
    auto Kacc = [&](int R, int c) { double s = 0; if (c < 0 || c >= L - 1) return s; for (int r = 0; r < R; ++r) s += (double)Jh[r * (L - 1) + c]; return s; };
    if (idx < p.n_gates) {
        const int g = p.gate_rc[idx], mirrored = (g >> 12) & 1, K = (g >> 13) & 7, low = (g >> 16) & 1;
        const int r = (g >> 6) & 63, c = g & 63;
        const double m = -2.0 * (double)Jv[(r - 1) * L + c];
        const double H = Hacc(r, c), Kl = Kacc(r, c - 1), Kr = Kacc(r, c);
        float* out = p.gate_k + (inst * p.n_gates + idx) * 8;
        if (g & GATE_RC_FLIP) {        // Z2 flip gate on column 0: kf[bit of column 1] = m - 2 K_0 sigma_1 (h = 0)
            out[0] = (float)(m - 2.0 * Kr); out[1] = (float)(m + 2.0 * Kr);
            for (int i = 2; i < 8; ++i) out[i] = 0.f;
        } else {
            // k[side][P bit][Q bit]: P = left neighbour in layout A, right neighbour in layout B
            float k[2][2][2];
            for (int np = 0; np < 2; ++np)
                for (int nq = 0; nq < 2; ++nq) {
                    const int nl = mirrored ? nq : np, nh = mirrored ? np : nq;
                    const double rho = H + (nl ? -Kl : Kl) + (nh ? -Kr : Kr);
                    k[0][np][nq] = (float)(m - 2.0 * rho);         // ka: a' = max(a, b + ka)
                    k[1][np][nq] = (float)(m + 2.0 * rho);         // kb: b' = max(b, a + kb)
                }
            const int pos = fused_chain_pos(low != 0, K);
            const int PN = pos == 0 ? -1 : fused_bit_of_digit(low != 0, 0, pos - 1);
            const int order = gate_order(K, PN);
            for (int np = 0; np < 2; ++np)
                for (int nq = 0; nq < 2; ++nq) {
                    if (order == ORDER_K0) { out[(np * 2 + nq) * 2] = k[1][np][nq]; out[(np * 2 + nq) * 2 + 1] = k[0][np][nq]; }
                    else if (order == ORDER_PN0) { out[nq * 2 + np] = k[0][np][nq]; out[4 + nq * 2 + np] = k[1][np][nq]; }
                    else { out[np * 2 + nq] = k[0][np][nq]; out[4 + np * 2 + nq] = k[1][np][nq]; }
                }
        }
    }
    if (idx < FFINAL_FLOATS) {
        float* out = p.final_tab + inst * FFINAL_FLOATS;
        if (idx < 512) {
            const int var = (int)idx >> 7, j = (int)idx & 127, tl = var & 1, th = var >> 1;
            const bool low = p.fin_low != 0;
            // register columns are consecutive: x0 .. x0+6
            const int d0 = low ? (p.fin_layout == 0 ? 0 : 5) : (p.fin_layout == 0 ? 0 : 2);
            const int x0 = p.col_off + p.fin_a + d0;
            double acc = 0;
            int bits[F_RB];
            for (int i = 0; i < F_RB; ++i) bits[i] = (j >> fused_bit_of_digit(low, p.fin_layout, d0 + i)) & 1;
            for (int i = 0; i < F_RB; ++i) {
                const int c = x0 + i;
                acc += bits[i] ? -Hacc(L, c) : Hacc(L, c);
                if (i + 1 < F_RB) acc += (bits[i] == bits[i + 1]) ? Kacc(L, c) : -Kacc(L, c);
            }
            acc += (tl == bits[0]) ? Kacc(L, x0 - 1) : -Kacc(L, x0 - 1);              // 0 when x0 = 0 (Z2: tl = 0 = sigma_0 up)
            acc += (th == bits[F_RB - 1]) ? Kacc(L, x0 + F_RB - 1) : -Kacc(L, x0 + F_RB - 1);   // 0 at the right edge
            out[idx] = (float)acc;
        } else if (idx < 576) {
            // per DIGIT of the kernel's index; Z2: digit 0 = column 1 also carries K_0 sigma_0 sigma_1 = K_0 sigma_1
            const int c = (int)idx - 512 + p.col_off;
            out[idx] = c < L ? (float)(Hacc(L, c) + (p.col_off && c == p.col_off ? Kacc(L, c - 1) : 0.0)) : 0.f;
        } else {
            const int c = (int)idx - 576 + p.col_off;
            out[idx] = c < L - 1 ? (float)Kacc(L, c) : 0.f;
        }
    }
}

}  // namespace ttn

namespace ttn {

// ---- S0 for Tropical<i16>: packed (lo = column-0 bit 0, hi = bit 1) gate constants and final table ------
// gate_rc: low << 16 | K << 13 | layout << 12 | r << 6 | c with c the lattice COLUMN; K = 7 is the
// gate on column 0 (the half of a word).  All values are integers (checked on the host).
__global__ void __launch_bounds__(256) fused16_prep_kernel(const FusedPrepParams p) {
    const unsigned long long inst = blockIdx.y;
    const int L = p.L;
    const float* Jh = p.Jh + inst * (unsigned long long)(L * (L - 1));
    const float* Jv = p.Jv + inst * (unsigned long long)((L - 1) * L);
    const float* hh = p.h ? p.h + inst * (unsigned long long)(L * L) : nullptr;
    const long idx = (long)blockIdx.x * blockDim.x + threadIdx.x;
    auto Hacc = [&](int R, int c) { double s = 0; if (hh) for (int r = 0; r < R; ++r) s += (double)hh[r * L + c]; return s; };
    auto Kacc = [&](int R, int c) { double s = 0; if (c < 0 || c >= L - 1) return s; for (int r = 0; r < R; ++r) s += (double)Jh[r * (L - 1) + c]; return s; };
    auto pack = [](double lo, double hi) { return ((unsigned)(int)lo & 0xffffu) | ((unsigned)(int)hi << 16); };
    if (idx < p.n_gates) {
        const int g = p.gate_rc[idx], mirrored = (g >> 12) & 1, K = (g >> 13) & 7;
        const int r = (g >> 6) & 63, c = g & 63;
        const double m = -2.0 * (double)Jv[(r - 1) * L + c];
        const double H = Hacc(r, c), Kl = Kacc(r, c - 1), Kr = Kacc(r, c);
        unsigned* out = reinterpret_cast<unsigned*>(p.gate_k) + (inst * p.n_gates + idx) * 8;
        auto kval = [&](int side, int nl, int nh) {
            const double rho = H + (nl ? -Kl : Kl) + (nh ? -Kr : Kr);
            return side == 0 ? m - 2.0 * rho : m + 2.0 * rho;
        };
        if (g & GATE_RC_FLIP) {       // Z2 flip gate on column 0; its neighbour bit (column 1) is the half itself
            for (int i = 0; i < 8; ++i) out[i] = 0u;
            out[0] = pack(m - 2.0 * Kr, m + 2.0 * Kr);
        } else if (K == 7) {          // the half column (0; Z2: 1, left neighbour sigma_0 = +1): kp[n] = (lo: ka, hi: kb),
            for (int i = 0; i < 8; ++i) out[i] = 0u;                  // n = bit of the next column
            for (int n = 0; n < 2; ++n) out[n] = pack(kval(0, 0, n), kval(1, 0, n));
        } else {
            for (int side = 0; side < 2; ++side)
                for (int np = 0; np < 2; ++np)
                    for (int nq = 0; nq < 2; ++nq) {
                        const int nl = mirrored ? nq : np, nh = mirrored ? np : nq;
                        // the column after the half column: the left neighbour is the half of the word itself
                        out[side * 4 + np * 2 + nq] = c == 1 + p.col_off ? pack(kval(side, 0, nh), kval(side, 1, nh))
                                                             : pack(kval(side, nl, nh), kval(side, nl, nh));
                    }
        }
    }
    if (idx < FFINAL_FLOATS) {
        float* out = p.final_tab + inst * FFINAL_FLOATS;
        if (idx < 512) {
            const int var = (int)idx >> 7, j = (int)idx & 127, tl = var & 1, th = var >> 1;
            const bool low = p.fin_low != 0;
            const int d0 = low ? (p.fin_layout == 0 ? 0 : 5) : (p.fin_layout == 0 ? 0 : 2);
            const int x0 = p.col_off + 1 + p.fin_a + d0;        // first register COLUMN (fin_a = word digit)
            int bits[F_RB];
            for (int i = 0; i < F_RB; ++i) bits[i] = (j >> fused_bit_of_digit(low, p.fin_layout, d0 + i)) & 1;
            double acc = 0;
            for (int i = 0; i < F_RB; ++i) {
                const int c = x0 + i;
                acc += bits[i] ? -Hacc(L, c) : Hacc(L, c);
                if (i + 1 < F_RB) acc += (bits[i] == bits[i + 1]) ? Kacc(L, c) : -Kacc(L, c);
            }
            acc += (th == bits[F_RB - 1]) ? Kacc(L, x0 + F_RB - 1) : -Kacc(L, x0 + F_RB - 1);
            const double kl = Kacc(L, x0 - 1);
            const int tl0 = x0 == 1 + p.col_off ? 0 : tl, tl1 = x0 == 1 + p.col_off ? 1 : tl;     // left neighbour = the half
            reinterpret_cast<unsigned*>(out)[idx] = pack(acc + ((tl0 == bits[0]) ? kl : -kl), acc + ((tl1 == bits[0]) ? kl : -kl));
        } else if (idx < 576) {
            // per DIGIT of the element index; Z2: digit 0 = column 1 also carries K_0 sigma_0 sigma_1 = K_0 sigma_1
            const int c = (int)idx - 512 + p.col_off;
            out[idx] = c < L ? (float)(Hacc(L, c) + (p.col_off && c == p.col_off ? Kacc(L, c - 1) : 0.0)) : 0.f;
        } else {
            const int c = (int)idx - 576 + p.col_off;
            out[idx] = c < L - 1 ? (float)Kacc(L, c) : 0.f;
        }
    }
}

}  // namespace ttn
