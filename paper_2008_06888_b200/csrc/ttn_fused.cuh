// ttn_fused.cuh -- fused register-phase pass kernel for the Ising Tropical<f32> sweep ("v3",
// diagonal frame; see planner.h for the frame and the schedule).
//
// One launch = one HBM pass.  Each WARP owns a tile of 2^12 state elements,
// 128 per thread, and runs the pass's micro-op program on it with no CTA-level cooperation:
//   * conjugated max-plus gates (A2) PAPER.md:242 on a register digit:
//         a' = max(a, b + ka[n]),  b' = max(b, a + kb[n]),   n = (bit c-1, bit c+1) of the index,
//     the row diagonals (A3), (A4) PAPER.md:247-252 folded into the 8 constants of the gate and
//     the common +Jv deferred to a scalar (ttn_api.cu): 1 FMNMX + 1/2 FADD2 per element;
//   * layout exchanges A <-> B through the warp's private shared-memory region with 128-bit,
//     bank-conflict-free accesses, synchronised with __syncwarp only;
//   * the last pass adds the accumulated diagonal A_{L-1}(s) (a 128-entry table over the
//     register digits in 4 boundary variants + a per-thread scalar) and max-reduces.
// Global traffic goes straight between HBM and registers: the LOW tile (columns 0..11) moves
// 128-byte lines; HIGH tiles (columns a..a+8 plus the riding columns 0..2 on the low lane bits)
// move whole 32-byte sectors, four per request.  The kernel is persistent (one CTA per SM);
// programs and gate constants are staged in shared memory once per launch and instance.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>
#include "planner.h"

namespace ttn {

// Warps per CTA (one CTA per SM).  The LOW kernel's global accesses need no address registers,
// so it fits 12 warps of 168 registers (3 per scheduler); the HIGH kernel keeps 8 warps of 255
// registers so that all 128 strided loads of a tile stay in flight.
constexpr int FWARPS_LOW = 12, FWARPS_HIGH = 8;
constexpr int FREGION_F4 = 33 * 32;       // float4 per warp exchange region (low tile: padded rows)
constexpr int FMAX_MOPS = 128;            // micro-ops per pass
constexpr int FMAX_GATES = 160;           // gates per pass (8 constants each)
constexpr int FFINAL_FLOATS = 4 * 128 + 2 * 64;   // final table (4 variants) + H[64] + K[64]
__host__ __device__ constexpr int fwarps(bool low) { return low ? FWARPS_LOW : FWARPS_HIGH; }
__host__ __device__ constexpr size_t fsmem_bytes(bool low) {
    return (size_t)fwarps(low) * FREGION_F4 * 16 + (size_t)FMAX_GATES * 32 + (size_t)FFINAL_FLOATS * 4 +
           (size_t)FMAX_MOPS * 4 + 64;
}

struct FusedParams {
    int L, a, low, flags, first_layout, last_layout, batch;
    float* state;                       // instance 0
    unsigned long long inst_stride;     // elements between instances
    unsigned long long tiles_per_inst;  // warp tiles (2^12 elements) per instance
    const MicroOp* mops; int n_mops;    // this pass's program
    const float* gate_k; int n_gates;   // [inst][all gates][8]; this pass's slice of instance 0
    unsigned long long gate_inst_stride;          // floats between instances
    const float* final_tab;             // [inst][FFINAL_FLOATS] (REDUCE pass only)
    float* part_x;                      // [batch][gridDim.x] (REDUCE)
    unsigned stagger_cycles;            // start delay per warp group (warp / 4), see the kernel
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

// ---- conjugated gate on register-index bit K ------------------------------------------------------
// NL / NH: register-index bit holding the left / right neighbour column, or -1 when that
// neighbour is constant per thread (its value is then tl / th).  k[0..3] = ka[nl][nh],
// k[4..7] = kb[nl][nh].
template <int K, int NL, int NH>
__device__ __forceinline__ void cgate(float (&v)[128], const float4 c0, const float4 c1, const int tl, const int th) {
    float ka[2][2] = {{c0.x, c0.y}, {c0.z, c0.w}}, kb[2][2] = {{c1.x, c1.y}, {c1.z, c1.w}};
    if (NL < 0) {
#pragma unroll
        for (int h = 0; h < 2; ++h) { ka[0][h] = tl ? ka[1][h] : ka[0][h]; kb[0][h] = tl ? kb[1][h] : kb[0][h]; }
    }
    if (NH < 0) {
#pragma unroll
        for (int l = 0; l < 2; ++l) { ka[l][0] = th ? ka[l][1] : ka[l][0]; kb[l][0] = th ? kb[l][1] : kb[l][0]; }
    }
    constexpr int B = 1 << K;
#define TTN_NL(j) (NL < 0 ? 0 : (((j) >> (NL < 0 ? 0 : NL)) & 1))
#define TTN_NH(j) (NH < 0 ? 0 : (((j) >> (NH < 0 ? 0 : NH)) & 1))
    if (K == 0) {
#pragma unroll
        for (int j = 0; j < 128; j += 2) {
            float t0, t1;     // t0 = a + kb (candidate for b), t1 = b + ka (candidate for a)
            add2(t0, t1, v[j], v[j + 1], kb[TTN_NL(j)][TTN_NH(j)], ka[TTN_NL(j)][TTN_NH(j)]);
            v[j] = fmaxf(v[j], t1);
            v[j + 1] = fmaxf(v[j + 1], t0);
        }
    } else {
#pragma unroll
        for (int j = 0; j < 128; j += 2) {
            if ((j & B) == 0) {
                float a0, a1, b0, b1;
                add2(a0, a1, v[j], v[j + 1], kb[TTN_NL(j)][TTN_NH(j)], kb[TTN_NL(j + 1)][TTN_NH(j + 1)]);
                add2(b0, b1, v[j + B], v[j + B + 1], ka[TTN_NL(j)][TTN_NH(j)], ka[TTN_NL(j + 1)][TTN_NH(j + 1)]);
                v[j] = fmaxf(v[j], b0); v[j + 1] = fmaxf(v[j + 1], b1);
                v[j + B] = fmaxf(v[j + B], a0); v[j + B + 1] = fmaxf(v[j + B + 1], a1);
            }
        }
    }
#undef TTN_NL
#undef TTN_NH
}

// register bit of the left / right neighbour of the digit held by register bit K (-1: per thread)
template <bool LOW, int LAYOUT, int K> struct Nbr {
    static constexpr int d = fused_digit_of_bit(LOW, LAYOUT, K);
    static constexpr int W = LOW ? F_WLOW : F_WHIGH;
    static constexpr int NL = d == 0 ? -1 : fused_bit_of_digit(LOW, LAYOUT, d - 1);
    static constexpr int NH = d == W - 1 ? -1 : fused_bit_of_digit(LOW, LAYOUT, d + 1);
};

// One round: for every set bit of `mask` (ascending) the next gate of that register digit.
template <bool LOW, int LAYOUT>
__device__ __forceinline__ void fround(float (&v)[128], const unsigned mask, const float4* __restrict__ gk,
                                       const int tl, const int th) {
#define TTN_G(Kk)                                                                                   \
    if (mask & (1u << Kk)) {                                                                        \
        const float4 c0 = gk[0], c1 = gk[1]; gk += 2;                                               \
        cgate<Kk, Nbr<LOW, LAYOUT, Kk>::NL, Nbr<LOW, LAYOUT, Kk>::NH>(v, c0, c1, tl, th);           \
    }
    TTN_G(0) TTN_G(1) TTN_G(2) TTN_G(3) TTN_G(4) TTN_G(5) TTN_G(6)
#undef TTN_G
}

// ---- exchange addressing: float4 index of register quad q for this lane -------------------------
//   LOW : chunk X = (d0..d4) + 32 (d7..d11), row-padded: f4 = X + (X >> 5)
//         A (lanes d7..d11): 33 lane + q          B (lanes d0..d4): lane + 33 q
//   HIGH: f4 = rho + 8 Y, Y = d0 + 2 d1 + 4 d4 + 8 d5 + 16 d6 + 32 d7 + 64 d8
//         A (lanes rho, d7, d8): rho + 256 (lane>>3) + 8 q      B (lanes rho, d0, d1): rho + 8 (lane>>3) + 32 q
template <bool LOW, int LAYOUT>
__device__ __forceinline__ int xbase(int lane) {
    if (LOW) return LAYOUT == 0 ? 33 * lane : lane;
    return LAYOUT == 0 ? (lane & 7) + 256 * (lane >> 3) : (lane & 7) + 8 * (lane >> 3);
}
template <bool LOW, int LAYOUT>
__device__ __forceinline__ constexpr int xstep() { return LOW ? (LAYOUT == 0 ? 1 : 33) : (LAYOUT == 0 ? 8 : 32); }

template <bool LOW, int LAYOUT>
__device__ __forceinline__ void xstore(const float (&v)[128], float4* reg, int lane) {
    float4* p = reg + xbase<LOW, LAYOUT>(lane);
#pragma unroll
    for (int q = 0; q < 32; ++q) p[q * xstep<LOW, LAYOUT>()] = make_float4(v[4 * q], v[4 * q + 1], v[4 * q + 2], v[4 * q + 3]);
}
template <bool LOW, int LAYOUT>
__device__ __forceinline__ void xload(float (&v)[128], const float4* reg, int lane) {
    const float4* p = reg + xbase<LOW, LAYOUT>(lane);
#pragma unroll
    for (int q = 0; q < 32; ++q) {
        const float4 t = p[q * xstep<LOW, LAYOUT>()];
        v[4 * q] = t.x; v[4 * q + 1] = t.y; v[4 * q + 2] = t.z; v[4 * q + 3] = t.w;
    }
}

// ---- global <-> register: element index e (inside the warp tile) of register j ---------------
//   LOW  B: e = lane + 32 j                      (address = tile base + e; 128 B per request)
//   HIGH A: e = 4 (j & 3) + ((j >> 2) & 3) + (j & 0x70) + 128 (lane >> 3)
//   HIGH B: e = (lane >> 3) + 4 j                (address = tile base + rho + (e << a))
__device__ __forceinline__ constexpr int ereg_high_a(int j) { return 4 * (j & 3) + ((j >> 2) & 3) + (j & 0x70); }

template <bool LOW, bool STORE>
__device__ __forceinline__ void gmove(float (&v)[128], float* tile, int lane, int layout, unsigned long long estride) {
    if (LOW) {
        float* p = tile + lane;                                   // layout B only (planner guarantees)
#pragma unroll
        for (int j = 0; j < 128; ++j) { if (STORE) p[32 * j] = v[j]; else v[j] = p[32 * j]; }
    } else if (layout == 0) {
        // 32-bit element offsets (e * 2^a < 2^32) keep the address math on the FMA pipe (IMAD.WIDE)
        const unsigned es = (unsigned)estride;
        float* p = tile + (lane & 7) + (unsigned long long)(128 * (lane >> 3)) * estride;
#pragma unroll
        for (int j = 0; j < 128; ++j) {
            float* q = p + (unsigned)(ereg_high_a(j)) * es;
            if (STORE) *q = v[j]; else v[j] = *q;
        }
    } else {
        const unsigned es = (unsigned)estride;
        float* p = tile + (lane & 7) + (unsigned long long)(lane >> 3) * estride;
#pragma unroll
        for (int j = 0; j < 128; ++j) {
            float* q = p + (unsigned)(4 * j) * es;
            if (STORE) *q = v[j]; else v[j] = *q;
        }
    }
}

// ---- last pass: v[j] += A_{L-1}(s) -------------------------------------------------------------------
// s_fin = [4 variants][128] table over the register digits (variant = tl + 2 th: the two boundary
// couplings to the per-thread neighbours) followed by H[64], K[64] (accumulated fields and
// horizontal couplings).  x0 = first register column; sthr = the element index with the register
// digits cleared.
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

template <bool LOW>
__global__ void __launch_bounds__(fwarps(LOW) * 32, 1) fused_pass_kernel(const FusedParams p) {
    constexpr int FWARPS = fwarps(LOW);
    extern __shared__ __align__(16) unsigned char fsm_raw[];
    float4* regions = reinterpret_cast<float4*>(fsm_raw);                              // FWARPS * FREGION_F4
    float4* s_gk = reinterpret_cast<float4*>(fsm_raw + (size_t)FWARPS * FREGION_F4 * 16);   // FMAX_GATES * 2
    float* s_fin = reinterpret_cast<float*>(s_gk + FMAX_GATES * 2);                     // FFINAL_FLOATS
    unsigned* s_mops = reinterpret_cast<unsigned*>(s_fin + FFINAL_FLOATS);              // FMAX_MOPS
    float* s_red = reinterpret_cast<float*>(s_mops + FMAX_MOPS);                        // FWARPS (<= 16)
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    float4* myreg = regions + warp * FREGION_F4;
    const unsigned long long gw = (unsigned long long)blockIdx.x * FWARPS + warp;
    const unsigned long long nw = (unsigned long long)gridDim.x * FWARPS;
    const unsigned long long estride = 1ull << p.a;

    // De-phase the warps of one scheduler (warps w, w+4, w+8 share SM sub-partition w % 4).  All
    // tiles cost the same and the schedulers share the alu pipe fairly, so warps that start
    // together stay in lock-step: they all compute, then all wait on memory, and the two never
    // overlap.  Starting group g one gate-phase later keeps one group in its memory phase while
    // the others compute.
    if (p.stagger_cycles && warp >= 4) {
        const long long t_end = clock64() + (long long)(warp >> 2) * p.stagger_cycles;
        while (clock64() < t_end) __nanosleep(256);
    }

    for (int inst = 0; inst < p.batch; ++inst) {
        // ---- stage this instance's program and gate constants (S0 outputs) into shared memory
        __syncthreads();
        for (int i = tid; i < p.n_mops; i += blockDim.x) {
            const MicroOp mo = p.mops[i];
            s_mops[i] = (unsigned)mo.code | ((unsigned)mo.mask << 8) | ((unsigned)mo.arg << 16);
        }
        {
            const float4* src = reinterpret_cast<const float4*>(p.gate_k + (size_t)inst * p.gate_inst_stride);
            for (int i = tid; i < p.n_gates * 2; i += blockDim.x) s_gk[i] = src[i];
        }
        if (p.flags & PASS_REDUCE)
            for (int i = tid; i < FFINAL_FLOATS; i += blockDim.x) s_fin[i] = p.final_tab[(size_t)inst * FFINAL_FLOATS + i];
        __syncthreads();
        float* S = p.state + (unsigned long long)inst * p.inst_stride;
        float wmax = -INFINITY;

        for (unsigned long long wt = gw; wt < p.tiles_per_inst; wt += nw) {
            // ---- tile geometry: base index, per-thread neighbour bits ------------------------------
            unsigned long long base;
            int tlA, thA, tlB, thB;     // per-thread left / right neighbour bit in layout A / B
            if (LOW) {
                base = wt << 12;
                tlA = 0;                                   // column -1 does not exist
                thA = lane & 1;                            // d7 (lane bit 0 in layout A)
                tlB = (lane >> 4) & 1;                     // d4 (lane bit 4 in layout B)
                thB = (p.L > F_WLOW) ? (int)(wt & 1ull) : 0;                      // column 12
            } else {
                const int amid = p.a - F_RIDE;
                const unsigned long long tmid = wt & ((1ull << amid) - 1), ttop = wt >> amid;
                base = (tmid << F_RIDE) + (ttop << (p.a + F_WHIGH));
                tlA = (int)((base >> (p.a - 1)) & 1ull);                          // column a-1 (>= 3)
                thA = (lane >> 3) & 1;                     // d7
                tlB = (lane >> 4) & 1;                     // d1
                thB = (p.a + F_WHIGH < p.L) ? (int)(ttop & 1ull) : 0;             // column a+9
            }
            float v[128];
            if (p.flags & PASS_INIT) {
#pragma unroll
                for (int j = 0; j < 128; ++j) v[j] = 0.f;                         // tropical one
            } else {
                gmove<LOW, false>(v, S + base, lane, p.first_layout, estride);
            }
            // ---- run the program ------------------------------------------------------------------
            int pc = 0, layout = p.first_layout;
            unsigned op = s_mops[0];
            for (;;) {
                const unsigned code = op & 0xffu;
                if (code == MC_END || code == MC_FINAL) break;
                const unsigned nxt = s_mops[pc + 1];
                if (code == MC_ROUND) {
                    const float4* gk = s_gk + 2 * (op >> 16);
                    if (layout == 0) fround<LOW, 0>(v, (op >> 8) & 0x7fu, gk, tlA, thA);
                    else fround<LOW, 1>(v, (op >> 8) & 0x7fu, gk, tlB, thB);
                } else if (code == MC_XAB) {
                    __syncwarp(); xstore<LOW, 0>(v, myreg, lane); __syncwarp(); xload<LOW, 1>(v, myreg, lane);
                    layout = 1;
                } else {
                    __syncwarp(); xstore<LOW, 1>(v, myreg, lane); __syncwarp(); xload<LOW, 0>(v, myreg, lane);
                    layout = 0;
                }
                op = nxt; ++pc;
            }
            // ---- store, or add A_{L-1}(s) and reduce ---------------------------------------------
            if (p.flags & PASS_REDUCE) {
                // element index with the register digits cleared, first register column, variant
                unsigned long long sthr; int x0, var;
                if (LOW) {
                    if (layout == 0) { sthr = base + ((unsigned long long)lane << 7); x0 = 0; var = tlA + 2 * thA; }
                    else { sthr = base + lane; x0 = 5; var = tlB + 2 * thB; }
                } else {
                    if (layout == 0) { sthr = base + (lane & 7) + ((unsigned long long)(lane >> 3) << (p.a + 7)); x0 = p.a; var = tlA + 2 * thA; }
                    else { sthr = base + (lane & 7) + ((unsigned long long)(lane >> 3) << p.a); x0 = p.a + 2; var = tlB + 2 * thB; }
                }
                const float cthr = final_thread_const(s_fin, p.L, x0, sthr);
                const float4* T = reinterpret_cast<const float4*>(s_fin + var * 128);
                float mx = -INFINITY;
#pragma unroll
                for (int q = 0; q < 32; ++q) {
                    const float4 t = T[q];
                    mx = fmaxf(mx, fmaxf(fmaxf(v[4 * q] + t.x, v[4 * q + 1] + t.y), fmaxf(v[4 * q + 2] + t.z, v[4 * q + 3] + t.w)));
                }
                wmax = fmaxf(wmax, mx + cthr);
            } else {
                gmove<LOW, true>(v, S + base, lane, p.last_layout, estride);
            }
        }
        if (p.flags & PASS_REDUCE) {
            for (int o = 16; o; o >>= 1) wmax = fmaxf(wmax, __shfl_xor_sync(0xffffffffu, wmax, o));
            if (lane == 0) s_red[warp] = wmax;
            __syncthreads();
            if (tid == 0) {
                float m = s_red[0];
                for (int w = 1; w < FWARPS; ++w) m = fmaxf(m, s_red[w]);
                p.part_x[(size_t)inst * gridDim.x + blockIdx.x] = m;
            }
        }
    }
}

// ---- S0: per-instance gate constants and the final table from the couplings ------------------------
struct FusedPrepParams {
    int L, n_gates;
    const int* gate_rc;            // [n_gates]  r * 64 + c
    const float* Jh; const float* Jv; const float* h;   // device couplings, per instance
    float* gate_k;                 // [inst][n_gates][8]
    float* final_tab;              // [inst][FFINAL_FLOATS]
    int fin_low, fin_layout, fin_a;   // tile kind, layout and start column of the last pass's end
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
        const int r = p.gate_rc[idx] >> 6, c = p.gate_rc[idx] & 63;
        const double m = -2.0 * (double)Jv[(r - 1) * L + c];
        const double H = Hacc(r, c), Kl = Kacc(r, c - 1), Kr = Kacc(r, c);
        float* out = p.gate_k + (inst * p.n_gates + idx) * 8;
        for (int nl = 0; nl < 2; ++nl)
            for (int nh = 0; nh < 2; ++nh) {
                const double rho = H + (nl ? -Kl : Kl) + (nh ? -Kr : Kr);
                out[nl * 2 + nh] = (float)(m - 2.0 * rho);         // ka: a' = max(a, b + ka)
                out[4 + nl * 2 + nh] = (float)(m + 2.0 * rho);     // kb: b' = max(b, a + kb)
            }
    }
    if (idx < FFINAL_FLOATS) {
        float* out = p.final_tab + inst * FFINAL_FLOATS;
        if (idx < 512) {
            const int var = (int)idx >> 7, j = (int)idx & 127, tl = var & 1, th = var >> 1;
            const bool low = p.fin_low != 0;
            const int W = low ? F_WLOW : F_WHIGH;
            // register columns are consecutive: x0 .. x0+6
            const int d0 = low ? (p.fin_layout == 0 ? 0 : 5) : (p.fin_layout == 0 ? 0 : 2);
            const int x0 = p.fin_a + d0;
            (void)W;
            double acc = 0;
            int bits[F_RB];
            for (int i = 0; i < F_RB; ++i) bits[i] = (j >> fused_bit_of_digit(low, p.fin_layout, d0 + i)) & 1;
            for (int i = 0; i < F_RB; ++i) {
                const int c = x0 + i;
                acc += bits[i] ? -Hacc(L, c) : Hacc(L, c);
                if (i + 1 < F_RB) acc += (bits[i] == bits[i + 1]) ? Kacc(L, c) : -Kacc(L, c);
            }
            acc += (tl == bits[0]) ? Kacc(L, x0 - 1) : -Kacc(L, x0 - 1);              // 0 when x0 = 0
            acc += (th == bits[F_RB - 1]) ? Kacc(L, x0 + F_RB - 1) : -Kacc(L, x0 + F_RB - 1);   // 0 at the right edge
            out[idx] = (float)acc;
        } else if (idx < 576) {
            const int c = (int)idx - 512;
            out[idx] = c < L ? (float)Hacc(L, c) : 0.f;
        } else {
            const int c = (int)idx - 576;
            out[idx] = c < L - 1 ? (float)Kacc(L, c) : 0.f;
        }
    }
}

}  // namespace ttn
