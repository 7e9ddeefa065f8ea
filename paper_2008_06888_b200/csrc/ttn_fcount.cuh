// ttn_fcount.cuh -- fused register-phase pass kernel for the Ising CountingTropical<f32,f64> sweep
// (energy + ground-state degeneracy, Eq. (4)), the counting sibling of
// ttn_fused.cuh: same diagonal frame, same mirrored layouts, same micro-op programs and planner
// (planner.h, GEOM_COUNT), with 32 elements (x f32, n f64) per thread instead of 128 floats.
//
//   warp tile = 2^10 elements.  LOW: columns 0..9 (4 KiB of x + 8 KiB of n, contiguous).
//   HIGH: 7 active columns a..a+6 + riding columns 0..2 on the low lane bits.
//   layout A: register bits 0..4 = tile digits 0..4, lanes = the rest
//   layout B: register bits 0..4 = tile digits W-1..W-5 (mirrored), lanes = digits 0..4 (LOW) /
//             riding + digits 0,1 (HIGH)
//   gate on register bit K, pair (a, b) = (bit clear, bit set), n = neighbour bits of the index:
//       ca = xb + ka[n], cb = xa + kb[n], ns = na + nb
//       na' = ca > xa ? nb : (ca == xa ? ns : na),   xa' = max(xa, ca)      (Eq. (4): ties add counts)
//       nb' = cb > xb ? na : (cb == xb ? ns : nb),   xb' = max(xb, cb)
// Exchanges go through the warp's private shared-memory region (x and n planes), conflict-free.
#pragma once
#include "ttn_fused.cuh"

namespace ttn {

constexpr int CRB = 5;                                   // register digits
constexpr int CW_LOW = 10, CW_HIGH = 7;
constexpr int CREGION_BYTES = 32 * 33 * 4 + 32 * 33 * 8; // padded x plane + padded n plane
// warps per CTA: 24x24 counting, batch 16, with 8 / 12 / 16 warps = 87.3 / 77.3 / 78.6 ms (profiles/r01m.md)
#ifndef TTN_CWARPS
#define TTN_CWARPS 12
#endif
constexpr int CWARPS = TTN_CWARPS;
constexpr int CFINAL_FLOATS = FFINAL_FLOATS;             // same table layout (first 4 x 32 entries used)
__host__ __device__ constexpr size_t csmem_bytes() {
    return (size_t)CWARPS * CREGION_BYTES + (size_t)(FMAX_GATES + 1) * 32 + (size_t)CFINAL_FLOATS * 4 +
           (size_t)FMAX_MOPS * 4 + 256;
}

struct CountParams {
    FusedParams f;                      // state = x plane; part_x, programs, constants as in the f32 kernel
    double* state_n;                    // n plane, instance 0
    double* part_n;                     // [batch][part_stride]
};

// 1.0 / 0.0 from a predicate: only the high word of the double is selected
__device__ __forceinline__ double ind(bool p) { return __hiloint2double(p ? 0x3ff00000 : 0, 0); }

// ---- counting gate on register bit K ------------------------------------------------------------------
template <int K, int PN, int QN>
__device__ __forceinline__ void cgate_count(float (&x)[32], double (&n)[32], const float4 c0, const float4 c1,
                                            const int tp, const int tq) {
    float ka[2][2] = {{c0.x, c0.y}, {c0.z, c0.w}}, kb[2][2] = {{c1.x, c1.y}, {c1.z, c1.w}};
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
    for (int j = 0; j < 32; ++j) {
        if (j & B) continue;
        const int np = PN < 0 ? 0 : (j >> (PN < 0 ? 0 : PN)) & 1, nq = QN < 0 ? 0 : (j >> (QN < 0 ? 0 : QN)) & 1;
        const float xa = x[j], xb = x[j + B];
        const double na = n[j], nb = n[j + B];
        const float ca = xb + ka[np][nq], cb = xa + kb[np][nq];
#ifdef TTN_COUNT_SELECT
        const double ns = na + nb;
        n[j] = ca > xa ? nb : (ca == xa ? ns : na);
        n[j + B] = cb > xb ? na : (cb == xb ? ns : nb);
#else
        // Eq. (4) as n' = n_keep [keep >= cand] + n_cand [cand >= keep] with 0/1 factors: the selects
        // of 64-bit counts (alu pipe, two per count) become one FP64 multiply-add each (exact: x 1, x 0)
        n[j] = fma(nb, ind(ca >= xa), na * ind(xa >= ca));
        n[j + B] = fma(na, ind(cb >= xb), nb * ind(xb >= cb));
#endif
        x[j] = fmaxf(xa, ca);
        x[j + B] = fmaxf(xb, cb);
    }
}

// register bit i = chain position i: P neighbour = bit i-1 (per thread for i = 0), Q = bit i+1
template <bool LOW>
__device__ __forceinline__ void cround(float (&x)[32], double (&n)[32], const unsigned mask,
                                       const float4* __restrict__& gk, const int tp, const int tq) {
#define TTN_CG(Kk)                                                                                 \
    if (mask & (1u << Kk)) {                                                                       \
        const float4 c0 = gk[0], c1 = gk[1]; gk += 2;                                              \
        cgate_count<Kk, Kk - 1, (Kk == CRB - 1 ? -1 : Kk + 1)>(x, n, c0, c1, tp, tq);              \
    }
    TTN_CG(0) TTN_CG(1) TTN_CG(2) TTN_CG(3) TTN_CG(4)
#undef TTN_CG
}

// ---- exchange planes -----------------------------------------------------------------------------------
// LOW: element (lo = d0..d4, hi = d5..d9) at index 33 lo + hi of a padded 32 x 33 plane.
//      A: lane = hi, register j = lo;   B: lane = lo, register j holds hi = rev5(j).
// HIGH: element (rho, d0..d6) at rho + 8 (d0^d5) + 16 (d1^d6) + 32 (d2 + 2 d3 + 4 d4 + 8 d5 + 16 d6).
//      A: lanes (rho, d5, d6), register j = d0..d4;   B: lanes (rho, d0, d1), register bits = d6,d5,d4,d3,d2.
template <bool LOW, int LAYOUT>
__device__ __forceinline__ int cx_index(int lane, int j) {
    if (LOW) return LAYOUT == 0 ? 33 * j + lane : 33 * lane + rev5(j);
    const int rho = lane & 7, l3 = (lane >> 3) & 1, l4 = (lane >> 4) & 1;
    if (LAYOUT == 0) {          // l3 = d5, l4 = d6
        const int d0 = j & 1, d1 = (j >> 1) & 1;
        return rho + 8 * (d0 ^ l3) + 16 * (d1 ^ l4) + 32 * (j >> 2) + 256 * l3 + 512 * l4;
    }
    // l3 = d0, l4 = d1; j bits: d6, d5, d4, d3, d2
    const int d6 = j & 1, d5 = (j >> 1) & 1, d4 = (j >> 2) & 1, d3 = (j >> 3) & 1, d2 = (j >> 4) & 1;
    return rho + 8 * (l3 ^ d5) + 16 * (l4 ^ d6) + 32 * (d2 + 2 * d3 + 4 * d4 + 8 * d5 + 16 * d6);
}
template <bool LOW, int LAYOUT, bool STORE>
__device__ __forceinline__ void cxmove(float (&x)[32], double (&n)[32], unsigned char* region, int lane) {
    float* px = reinterpret_cast<float*>(region);
    double* pn = reinterpret_cast<double*>(region + 32 * 33 * 4);
#pragma unroll
    for (int j = 0; j < 32; ++j) {
        const int i = cx_index<LOW, LAYOUT>(lane, j);
        if (STORE) { px[i] = x[j]; pn[i] = n[j]; } else { x[j] = px[i]; n[j] = pn[i]; }
    }
}

// ---- Z2 flip gate (h = 0; planner.h "GLOBAL-FLIP (Z2) REDUCTION"), counting form --------------------------
//     c = x[~u] + kf[bit of column 1 in u];   n'[u] = n[u] [x >= c] + n[~u] [c >= x];   x'[u] = max(x[u], c)
// ~u = register 31 - j of lane 31 - lane of the partner warp (warp ^ 1), which holds the complement
// tile in the same layout; both warps publish (x, n) in their own exchange region first.
template <int LAYOUT>
__device__ __forceinline__ void cflipgate(float (&x)[32], double (&n)[32], unsigned char* myreg, const unsigned char* preg,
                                          const int lane, const int warp, const float k0, const float k1) {
    __syncwarp();
    cxmove<true, LAYOUT, true>(x, n, myreg, lane);
    pair_sync(warp);
    const float* px = reinterpret_cast<const float*>(preg);
    const double* pn = reinterpret_cast<const double*>(preg + 32 * 33 * 4);
    // column 1 = tile digit 0: register bit 0 in layout A, lane bit 0 in layout B
    const float kl = (lane & 1) ? k1 : k0;
#pragma unroll
    for (int j = 0; j < 32; ++j) {
        const int i = cx_index<true, LAYOUT>(31 - lane, 31 - j);
        const float c = px[i] + (LAYOUT == 0 ? ((j & 1) ? k1 : k0) : kl);
        const double m = pn[i];
        n[j] = fma(m, ind(c >= x[j]), n[j] * ind(x[j] >= c));
        x[j] = fmaxf(x[j], c);
    }
    pair_sync(warp);
}

// ---- global <-> register ----------------------------------------------------------------------------
//   LOW  B: e = lane + 32 rev5(j)
//   HIGH A: e = j + 32 (lane >> 3);   HIGH B: e = (lane >> 3) + 4 rev5(j);   address = tile + rho + (e << a)
template <bool LOW, int LAYOUT, bool STORE>
__device__ __forceinline__ void cgmove(float (&x)[32], double (&n)[32], float* tx, double* tn, int lane,
                                       unsigned sb, int a) {
    if (LOW) {
        float* px = tx + lane; double* pn = tn + lane;
#pragma unroll
        for (int j = 0; j < 32; ++j) {
            if (STORE) { px[32 * rev5(j)] = x[j]; pn[32 * rev5(j)] = n[j]; }
            else { x[j] = px[32 * rev5(j)]; n[j] = pn[32 * rev5(j)]; }
        }
        return;
    }
    const unsigned elane = (LAYOUT == 0) ? 32u * (unsigned)(lane >> 3) : (unsigned)(lane >> 3);
    const unsigned long long off = (unsigned long long)(lane & 7) + ((unsigned long long)elane << a);
    const unsigned long long gx = (unsigned long long)__cvta_generic_to_global(tx + off);
    const unsigned long long gn = (unsigned long long)__cvta_generic_to_global(tn + off);
#pragma unroll
    for (int j = 0; j < 32; ++j) {
        const unsigned e = LAYOUT == 0 ? (unsigned)j : 4u * (unsigned)rev5(j);
        const unsigned long long qx = addr_mad(gx, sb, e), qn = addr_mad(gn, 2u * sb, e);
        if (STORE) {
            stg_f32(qx, x[j]);
            asm volatile("st.global.f64 [%0], %1;" :: "l"(qn), "d"(n[j]) : "memory");
        } else {
            x[j] = ldg_f32(qx);
            asm volatile("ld.global.f64 %0, [%1];" : "=d"(n[j]) : "l"(qn));
        }
    }
}

__device__ __forceinline__ float cfinal_thread_const(const float* s_fin, int L, int x0, unsigned long long sthr) {
    const float* H = s_fin + 512; const float* Kc = s_fin + 576;
    float acc = 0.f;
    for (int c = 0; c < L; ++c) {
        const bool in_r = (c >= x0 && c < x0 + CRB);
        const int bc = (int)((sthr >> c) & 1ull);
        if (!in_r) acc += bc ? -H[c] : H[c];
        if (c + 1 < L) {
            const bool in_r1 = (c + 1 >= x0 && c + 1 < x0 + CRB);
            if (!in_r && !in_r1) {
                const int b1 = (int)((sthr >> (c + 1)) & 1ull);
                acc += (bc == b1) ? Kc[c] : -Kc[c];
            }
        }
    }
    return acc;
}

// Z2 (LOW only): flip-reduced state, warp pairs on tiles (T, ~T), flip gates (ttn_fused.cuh)
template <bool LOW, bool Z2 = false>
__global__ void __launch_bounds__(CWARPS * 32, 1) fcount_pass_kernel(const CountParams cp) {
    const FusedParams& p = cp.f;
    extern __shared__ __align__(16) unsigned char csm_raw[];
    unsigned char* regions = csm_raw;                                                        // CWARPS * CREGION_BYTES
    float4* s_gk = reinterpret_cast<float4*>(csm_raw + (size_t)CWARPS * CREGION_BYTES);     // (FMAX_GATES + 1) * 2
    float* s_fin = reinterpret_cast<float*>(s_gk + (FMAX_GATES + 1) * 2);
    unsigned* s_mops = reinterpret_cast<unsigned*>(s_fin + CFINAL_FLOATS);
    float* s_redx = reinterpret_cast<float*>(s_mops + FMAX_MOPS);                            // CWARPS
    double* s_redn = reinterpret_cast<double*>(s_redx + 16);                                 // CWARPS
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    unsigned char* myreg = regions + (size_t)warp * CREGION_BYTES;
    const unsigned long long gw = p.cta_per_inst ? (unsigned long long)warp : (unsigned long long)blockIdx.x * CWARPS + warp;
    const unsigned long long nw = p.cta_per_inst ? (unsigned long long)CWARPS : (unsigned long long)gridDim.x * CWARPS;
    constexpr int W = LOW ? CW_LOW : CW_HIGH;

    for (int inst = p.cta_per_inst ? (int)blockIdx.x : 0; inst < p.batch; inst += p.cta_per_inst ? (int)gridDim.x : 1) {
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
            for (int i = tid; i < CFINAL_FLOATS; i += blockDim.x) s_fin[i] = p.final_tab[(size_t)inst * CFINAL_FLOATS + i];
        __syncthreads();
        float* SX = p.state + (unsigned long long)inst * p.inst_stride;
        double* SN = cp.state_n + (unsigned long long)inst * p.inst_stride;
        float wmax = -INFINITY; double wcnt = 0.0;

        for (unsigned long long it = 0;; ++it) {
            unsigned long long wt;
            if (LOW && Z2) {                               // the pair (2k, 2k + 1) takes tile t and its complement
                const unsigned long long t = it * (nw >> 1) + (gw >> 1);
                if (t >= (p.tiles_per_inst >> 1)) break;
                wt = (gw & 1ull) ? p.tiles_per_inst - 1 - t : t;
            } else {
                wt = LOW ? it * nw + gw : 4ull * (it * (nw >> 2) + (gw >> 2)) + (unsigned long long)(warp & 3);
                if ((LOW ? wt : (wt & ~3ull)) >= p.tiles_per_inst) break;
            }
            if (!LOW && wt >= p.tiles_per_inst) {          // partial last group: keep the barrier counts equal
                if (!(p.flags & PASS_INIT)) group_sync(warp);
                if (!(p.flags & PASS_REDUCE)) group_sync(warp);
                continue;
            }
            unsigned long long base;
            int tpA, tqA, tpB, tqB;
            if (LOW) {
                base = wt << CW_LOW;
                tpA = 0;                                   // column -1 does not exist
                tqA = lane & 1;                            // d5
                tpB = (p.L > CW_LOW) ? (int)(wt & 1ull) : 0;   // column 10
                tqB = (lane >> 4) & 1;                     // d4
            } else {
                const int amid = p.a - F_RIDE;
                const unsigned long long tmid = wt & ((1ull << amid) - 1), ttop = wt >> amid;
                base = (tmid << F_RIDE) + (ttop << (p.a + CW_HIGH));
                tpA = (int)((base >> (p.a - 1)) & 1ull);   // column a-1
                tqA = (lane >> 3) & 1;                     // d5
                tpB = (p.a + CW_HIGH < p.L) ? (int)(ttop & 1ull) : 0;   // column a+7
                tqB = (lane >> 4) & 1;                     // d1
            }
            float x[32]; double n[32];
            if (p.flags & PASS_INIT) {
#pragma unroll
                for (int j = 0; j < 32; ++j) { x[j] = 0.f; n[j] = 1.0; }          // counting one = (0, 1)
            } else {
                if (!LOW) group_sync(warp);
                if (LOW || p.first_layout == 1) cgmove<LOW, 1, false>(x, n, SX + base, SN + base, lane, p.stride_bytes, p.a);
                else cgmove<LOW, 0, false>(x, n, SX + base, SN + base, lane, p.stride_bytes, p.a);
            }
            int pc = 0, layout = p.first_layout;
            unsigned op = s_mops[0];
            for (;;) {
                const unsigned code = op & 0xffu;
                if (code == MC_END || code == MC_FINAL) break;
                const unsigned nxt = s_mops[pc + 1];
                if (code == MC_ROUND) {
                    const float4* gk = s_gk + 2 * ((op >> 16) & 0x7fffu);
                    cround<LOW>(x, n, (op >> 8) & 0x1fu, gk, layout ? tpB : tpA, layout ? tqB : tqA);
                    if (LOW && Z2 && (op >> 31)) {         // the round ends with the flip gate (column 0)
                        const float4 kf = gk[0];
                        const unsigned char* preg = regions + (size_t)(warp ^ 1) * CREGION_BYTES;
                        if (layout == 0) cflipgate<0>(x, n, myreg, preg, lane, warp, kf.x, kf.y);
                        else cflipgate<1>(x, n, myreg, preg, lane, warp, kf.x, kf.y);
                    }
                } else if (code == MC_XAB) {
                    __syncwarp(); cxmove<LOW, 0, true>(x, n, myreg, lane); __syncwarp(); cxmove<LOW, 1, false>(x, n, myreg, lane);
                    layout = 1;
                } else {
                    __syncwarp(); cxmove<LOW, 1, true>(x, n, myreg, lane); __syncwarp(); cxmove<LOW, 0, false>(x, n, myreg, lane);
                    layout = 0;
                }
                op = nxt; ++pc;
            }
            if (p.flags & PASS_REDUCE) {
                unsigned long long sthr; int x0, var;
                if (LOW) {
                    if (layout == 0) { sthr = base + ((unsigned long long)lane << CRB); x0 = 0; var = tpA + 2 * tqA; }
                    else { sthr = base + lane; x0 = CW_LOW - CRB; var = tqB + 2 * tpB; }
                } else {
                    if (layout == 0) { sthr = base + (lane & 7) + ((unsigned long long)(lane >> 3) << (p.a + CRB)); x0 = p.a; var = tpA + 2 * tqA; }
                    else { sthr = base + (lane & 7) + ((unsigned long long)(lane >> 3) << p.a); x0 = p.a + CW_HIGH - CRB; var = tqB + 2 * tpB; }
                }
                const float cthr = cfinal_thread_const(s_fin, p.L, x0, sthr);
                const float* T = s_fin + var * 32;
                float mx = -INFINITY;
#pragma unroll
                for (int j = 0; j < 32; ++j) { x[j] = (x[j] + T[j]) + cthr; mx = fmaxf(mx, x[j]); }
                for (int o = 16; o; o >>= 1) mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, o));
                double cnt = 0.0;
#pragma unroll
                for (int j = 0; j < 32; ++j) if (x[j] == mx) cnt += n[j];
                for (int o = 16; o; o >>= 1) cnt += __shfl_xor_sync(0xffffffffu, cnt, o);
                if (mx > wmax) { wmax = mx; wcnt = cnt; } else if (mx == wmax) { wcnt += cnt; }
            } else {
                if (!LOW) group_sync(warp);
                if (LOW || p.last_layout == 1) cgmove<LOW, 1, true>(x, n, SX + base, SN + base, lane, p.stride_bytes, p.a);
                else cgmove<LOW, 0, true>(x, n, SX + base, SN + base, lane, p.stride_bytes, p.a);
            }
        }
        if (p.flags & PASS_REDUCE) {
            if (lane == 0) { s_redx[warp] = wmax; s_redn[warp] = wcnt; }
            __syncthreads();
            if (tid == 0) {
                float m = s_redx[0];
                for (int w = 1; w < CWARPS; ++w) m = fmaxf(m, s_redx[w]);
                double c = 0.0;
                for (int w = 0; w < CWARPS; ++w) if (s_redx[w] == m) c += s_redn[w];
                const size_t slot = (size_t)inst * p.part_stride + (p.cta_per_inst ? 0 : blockIdx.x);
                p.part_x[slot] = m; cp.part_n[slot] = c;
            }
        }
        (void)W;
    }
}

// ---- S0: gate constants k[side][P][Q] and the final table (4 variants x 32) + H, K -------------------------
struct CountPrepParams {
    int L, n_gates;
    const int* gate_rc;            // low << 16 | K << 13 | layout << 12 | r << 6 | c
    const float* Jh; const float* Jv; const float* h;
    float* gate_k;                 // [inst][n_gates][8]
    float* final_tab;              // [inst][CFINAL_FLOATS]
    int fin_low, fin_layout, fin_a;
    int col_off;                   // Z2: 1 = the kernel's digit d is lattice column d + 1 (fin_a is a digit)
};

__global__ void __launch_bounds__(256) fcount_prep_kernel(const CountPrepParams p) {
    const unsigned long long inst = blockIdx.y;
    const int L = p.L;
    const float* Jh = p.Jh + inst * (unsigned long long)(L * (L - 1));
    const float* Jv = p.Jv + inst * (unsigned long long)((L - 1) * L);
    const float* hh = p.h ? p.h + inst * (unsigned long long)(L * L) : nullptr;
    const long idx = (long)blockIdx.x * blockDim.x + threadIdx.x;
    auto Hacc = [&](int R, int c) { double s = 0; if (hh) for (int r = 0; r < R; ++r) s += (double)hh[r * L + c]; return s; };
    auto Kacc = [&](int R, int c) { double s = 0; if (c < 0 || c >= L - 1) return s; for (int r = 0; r < R; ++r) s += (double)Jh[r * (L - 1) + c]; return s; };
    if (idx < p.n_gates) {
        const int g = p.gate_rc[idx], mirrored = (g >> 12) & 1, r = (g >> 6) & 63, c = g & 63;
        const double m = -2.0 * (double)Jv[(r - 1) * L + c];
        const double H = Hacc(r, c), Kl = Kacc(r, c - 1), Kr = Kacc(r, c);
        float* out = p.gate_k + (inst * p.n_gates + idx) * 8;
        if (g & GATE_RC_FLIP) {        // Z2 flip gate on column 0: kf[bit of column 1] = m - 2 K_0 sigma_1 (h = 0)
            out[0] = (float)(m - 2.0 * Kr); out[1] = (float)(m + 2.0 * Kr);
            for (int i = 2; i < 8; ++i) out[i] = 0.f;
        } else {
            for (int np = 0; np < 2; ++np)
                for (int nq = 0; nq < 2; ++nq) {
                    const int nl = mirrored ? nq : np, nh = mirrored ? np : nq;      // P = left in A, right in B
                    const double rho = H + (nl ? -Kl : Kl) + (nh ? -Kr : Kr);
                    out[np * 2 + nq] = (float)(m - 2.0 * rho);
                    out[4 + np * 2 + nq] = (float)(m + 2.0 * rho);
                }
        }
    }
    if (idx < CFINAL_FLOATS) {
        float* out = p.final_tab + inst * CFINAL_FLOATS;
        if (idx < 128) {
            const int var = (int)idx >> 5, j = (int)idx & 31, tl = var & 1, th = var >> 1;
            const int Wt = p.fin_low ? CW_LOW : CW_HIGH;
            const int x0 = p.col_off + p.fin_a + (p.fin_layout == 0 ? 0 : Wt - CRB);       // first register column
            int bits[CRB];
            for (int i = 0; i < CRB; ++i) bits[i] = (j >> (p.fin_layout == 0 ? i : CRB - 1 - i)) & 1;
            double acc = 0;
            for (int i = 0; i < CRB; ++i) {
                const int c = x0 + i;
                acc += bits[i] ? -Hacc(L, c) : Hacc(L, c);
                if (i + 1 < CRB) acc += (bits[i] == bits[i + 1]) ? Kacc(L, c) : -Kacc(L, c);
            }
            acc += (tl == bits[0]) ? Kacc(L, x0 - 1) : -Kacc(L, x0 - 1);
            acc += (th == bits[CRB - 1]) ? Kacc(L, x0 + CRB - 1) : -Kacc(L, x0 + CRB - 1);
            out[idx] = (float)acc;
        } else if (idx >= 512 && idx < 576) {
            // per DIGIT of the kernel's index; Z2: digit 0 = column 1 also carries K_0 sigma_0 sigma_1 = K_0 sigma_1
            const int c = (int)idx - 512 + p.col_off;
            out[idx] = c < L ? (float)(Hacc(L, c) + (p.col_off && c == p.col_off ? Kacc(L, c - 1) : 0.0)) : 0.f;
        } else if (idx >= 576) {
            const int c = (int)idx - 576 + p.col_off;
            out[idx] = c < L - 1 ? (float)Kacc(L, c) : 0.f;
        } else out[idx] = 0.f;
    }
}

}  // namespace ttn
