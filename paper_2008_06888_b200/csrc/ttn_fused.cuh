// ttn_fused.cuh -- fused register-phase pass kernel for the Ising Tropical<f32> sweep ("v2").
//
// One launch = one HBM pass.  Each WARP owns a tile of 11 active digits
// [a, a+11) of the state index = 2^11 elements, 64 per thread, and runs the pass's micro-op
// program (planner.h, FusedPlan) on it:
//   * max-plus gates (A2) PAPER.md:242 on a register digit:  v[j] = max(v[j], v[j ^ bit] + m),
//     m = -2 J, the common +J deferred to a scalar (ttn_api.cu) -- 1 FMNMX + 1/2 FADD2 per element;
//   * diagonal gates (A3), (A4) PAPER.md:247-252 as 64-entry tables: v[j] += T[j];
//   * layout exchanges (register digits d0..d5 <-> d5..d10) through the warp's private,
//     padded shared-memory region, synchronised with __syncwarp only.
// Global <-> shared staging is CTA-wide and coalesced: the low tile (a = 0) moves contiguous
// 8 KiB per warp with 128-bit accesses; high tiles move 32-byte runs (3 riding digits), one
// riding value per warp.  The kernel is persistent (grid = resident CTAs), so programs and
// tables stay in shared memory / L1 across tiles.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>
#include "planner.h"

namespace ttn {

constexpr int FW = 11;                 // active digits per warp tile
constexpr int FWARPS = 8;              // warps per CTA = 2^ride
constexpr int FRIDE = 3;
constexpr int FROW = 68;               // padded row: 64 elements + 4 words
constexpr int FREGION = 32 * FROW + 4; // words per warp region (2180: == 4 mod 8, see staging)
constexpr int FMAX_MOPS = 512;
constexpr int FMAX_GATES = 256;

struct FusedParams {
    int L, a, ride, flags;
    float* state;                       // instance 0
    unsigned long long inst_stride;     // elements between instances
    unsigned long long tiles_per_inst;  // CTA tiles (2^14 elements) per instance
    unsigned long long total_tiles;     // tiles_per_inst * batch
    const MicroOp* mops; int n_mops;    // this pass's program
    const float* gate_m; int n_gates; int gate_inst_stride;       // this pass's slice, instance 0
    const float* tables; unsigned long long table_inst_stride;    // this pass's slice, instance 0
    float* part_x;                      // [total_tiles] (REDUCE)
};

__device__ __forceinline__ int fpad(int e) { return e + 4 * (e >> 6); }

// ---- gate on register bit K: v[j] <- max(v[j], v[j^bit] + m) -----------------------------------
template <int K>
__device__ __forceinline__ void fgate(float (&v)[64], const float m) {
    constexpr int B = 1 << K;
    if (K == 0) {
#pragma unroll
        for (int j = 0; j < 64; j += 2) {
            float t0 = v[j] + m, t1 = v[j + 1] + m;
            v[j] = fmaxf(v[j], t1);
            v[j + 1] = fmaxf(v[j + 1], t0);
        }
    } else {
#pragma unroll
        for (int j = 0; j < 64; ++j) {
            if ((j & B) == 0 && (j & 1) == 0) {
                float a0 = v[j] + m, a1 = v[j + 1] + m;
                float b0 = v[j + B] + m, b1 = v[j + B + 1] + m;
                v[j] = fmaxf(v[j], b0); v[j + 1] = fmaxf(v[j + 1], b1);
                v[j + B] = fmaxf(v[j + B], a0); v[j + B + 1] = fmaxf(v[j + B + 1], a1);
            }
        }
    }
}

__device__ __forceinline__ void ftable(float (&v)[64], const float4* __restrict__ T) {
#pragma unroll
    for (int q = 0; q < 16; ++q) {
        float4 t = __ldg(T + q);
        v[4 * q] += t.x; v[4 * q + 1] += t.y; v[4 * q + 2] += t.z; v[4 * q + 3] += t.w;
    }
}

// layout A: thread = row `lane` (digits d6..d10), registers = 64 consecutive words of the row
__device__ __forceinline__ void fload_a(float (&v)[64], const float* reg, int lane) {
    const float4* p = reinterpret_cast<const float4*>(reg + FROW * lane);
#pragma unroll
    for (int q = 0; q < 16; ++q) { float4 t = p[q]; v[4 * q] = t.x; v[4 * q + 1] = t.y; v[4 * q + 2] = t.z; v[4 * q + 3] = t.w; }
}
__device__ __forceinline__ void fstore_a(const float (&v)[64], float* reg, int lane) {
    float4* p = reinterpret_cast<float4*>(reg + FROW * lane);
#pragma unroll
    for (int q = 0; q < 16; ++q) p[q] = make_float4(v[4 * q], v[4 * q + 1], v[4 * q + 2], v[4 * q + 3]);
}
// layout B: thread = digits d0..d4 = lane, register j = digits d5..d10: element lane + 32 j
__device__ __forceinline__ void fload_b(float (&v)[64], const float* reg, int lane) {
#pragma unroll
    for (int j = 0; j < 64; ++j) v[j] = reg[lane + 32 * j + 4 * (j >> 1)];
}
__device__ __forceinline__ void fstore_b(const float (&v)[64], float* reg, int lane) {
#pragma unroll
    for (int j = 0; j < 64; ++j) reg[lane + 32 * j + 4 * (j >> 1)] = v[j];
}

__global__ void __launch_bounds__(FWARPS * 32, 2) fused_pass_kernel(const FusedParams p) {
    extern __shared__ __align__(16) float fsm[];
    float* regions = fsm;                                         // FWARPS * FREGION
    float* s_m = fsm + FWARPS * FREGION;                          // FMAX_GATES
    MicroOp* s_mops = reinterpret_cast<MicroOp*>(s_m + FMAX_GATES);   // FMAX_MOPS
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    float* myreg = regions + warp * FREGION;

    for (int i = tid; i < p.n_mops; i += blockDim.x) s_mops[i] = p.mops[i];
    unsigned long long cur_inst = ~0ull;

    for (unsigned long long gt = blockIdx.x; gt < p.total_tiles; gt += gridDim.x) {
        const unsigned long long inst = gt / p.tiles_per_inst;
        const unsigned long long tile = gt % p.tiles_per_inst;
        float* S = p.state + inst * p.inst_stride;
        if (inst != cur_inst) {                                   // (re)load this instance's gate constants
            __syncthreads();
            for (int i = tid; i < p.n_gates; i += blockDim.x) s_m[i] = p.gate_m[inst * p.gate_inst_stride + i];
            cur_inst = inst;
        }
        // ---- tile geometry ----------------------------------------------------------------------
        unsigned long long base;       // global index of (riding 0, e = 0)
        unsigned long long wbase;      // global index of this warp's element e = 0
        if (p.ride == 0) { base = tile << 14; wbase = base + ((unsigned long long)warp << FW); }
        else {
            const int amid = p.a - FRIDE;
            const unsigned long long tmid = tile & ((1ull << amid) - 1), ttop = tile >> amid;
            base = (tmid << FRIDE) + (ttop << (p.a + FW));
            wbase = base + warp;
        }
        // ---- stage in ----------------------------------------------------------------------------
        if (p.flags & PASS_INIT) {
            for (int i = tid; i < FWARPS * FREGION; i += blockDim.x) regions[i] = 0.f;
        } else if (p.ride == 0) {
            const float4* g = reinterpret_cast<const float4*>(S + base);
#pragma unroll 4
            for (int i = 0; i < 16; ++i) {
                int f = i * 256 + tid;                            // float4 index in the CTA tile
                float4 t = g[f];
                int wt = f >> 9, e = (f & 511) << 2;
                *reinterpret_cast<float4*>(regions + wt * FREGION + fpad(e)) = t;
            }
        } else {
            const unsigned long long estride = 1ull << p.a;
#pragma unroll 4
            for (int i = 0; i < 16; ++i) {
                int f = i * 256 + tid;                            // run e = f >> 1, half = f & 1
                int e = f >> 1, half = f & 1;
                float4 t = *reinterpret_cast<const float4*>(S + base + (unsigned long long)e * estride + 4 * half);
                float* r0 = regions + (4 * half) * FREGION + fpad(e);
                r0[0] = t.x; r0[FREGION] = t.y; r0[2 * FREGION] = t.z; r0[3 * FREGION] = t.w;
            }
        }
        __syncthreads();

        // ---- run the program on this warp's tile --------------------------------------------------
        {
            const int vA = (p.a > 0) ? (int)((wbase >> (p.a - 1)) & 1ull) : 0;          // outer neighbour a-1
            const int vB = (p.a + FW < p.L) ? (int)((wbase >> (p.a + FW)) & 1ull) : 0;  // outer neighbour a+W
            const float* tabs = p.tables + inst * p.table_inst_stride;
            float v[64];
#pragma unroll
            for (int j = 0; j < 64; ++j) v[j] = 0.f;
            int pc = 0;
            MicroOp op = s_mops[0];
            float m = s_m[op.arg & (FMAX_GATES - 1)];
            for (;;) {
                if (op.code == MC_END) break;
                const MicroOp nxt = s_mops[pc + 1];
                const float nm = s_m[nxt.arg & (FMAX_GATES - 1)];
                switch (op.code) {
                    case MC_LOAD_A: __syncwarp(); fload_a(v, myreg, lane); break;
                    case MC_LOAD_B: __syncwarp(); fload_b(v, myreg, lane); break;
                    case MC_STORE_A: fstore_a(v, myreg, lane); break;
                    case MC_STORE_B: fstore_b(v, myreg, lane); break;
                    case MC_TABLE: {
                        // table index op.arg, layout in op.k (0 = A: variant vA, 1 = B: variant vB)
                        const int var = op.k ? vB : vA;
                        ftable(v, reinterpret_cast<const float4*>(tabs + ((size_t)op.arg * 2 + var) * 64));
                        break;
                    }
                    case MC_GATE:
                        switch (op.k) {
                            case 0: fgate<0>(v, m); break;
                            case 1: fgate<1>(v, m); break;
                            case 2: fgate<2>(v, m); break;
                            case 3: fgate<3>(v, m); break;
                            case 4: fgate<4>(v, m); break;
                            default: fgate<5>(v, m); break;
                        }
                        break;
                    default: break;
                }
                op = nxt; m = nm; ++pc;
            }
        }
        __syncthreads();

        // ---- stage out / reduce ------------------------------------------------------------------
        if (p.flags & PASS_REDUCE) {
            float mx = -INFINITY;
            for (int i = tid; i < FWARPS * 2048; i += blockDim.x) mx = fmaxf(mx, regions[(i >> 11) * FREGION + fpad(i & 2047)]);
            for (int o = 16; o; o >>= 1) mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, o));
            __shared__ float red[FWARPS];
            if (lane == 0) red[warp] = mx;
            __syncthreads();
            if (tid == 0) { float b = red[0]; for (int w = 1; w < FWARPS; ++w) b = fmaxf(b, red[w]); p.part_x[gt] = b; }
        } else if (p.ride == 0) {
            float4* g = reinterpret_cast<float4*>(S + base);
#pragma unroll 4
            for (int i = 0; i < 16; ++i) {
                int f = i * 256 + tid;
                int wt = f >> 9, e = (f & 511) << 2;
                g[f] = *reinterpret_cast<const float4*>(regions + wt * FREGION + fpad(e));
            }
        } else {
            const unsigned long long estride = 1ull << p.a;
#pragma unroll 4
            for (int i = 0; i < 16; ++i) {
                int f = i * 256 + tid;
                int e = f >> 1, half = f & 1;
                const float* r0 = regions + (4 * half) * FREGION + fpad(e);
                float4 t = make_float4(r0[0], r0[FREGION], r0[2 * FREGION], r0[3 * FREGION]);
                *reinterpret_cast<float4*>(S + base + (unsigned long long)e * estride + 4 * half) = t;
            }
        }
        __syncthreads();
    }
}

// ---- S0: per-instance gate constants and diagonal tables from the couplings ----------------------
struct FusedPrepParams {
    int L, n_gates, n_tables;
    const int* gate_jv;            // [n_gates]
    const FusedTable* tables;      // [n_tables]
    const TableTerm* terms;
    const float* Jh; const float* Jv; const float* h;   // device couplings, per instance
    float* gate_m;                 // [inst][n_gates]
    float* table_out;              // [inst][n_tables][2][64]
};

__global__ void __launch_bounds__(256) fused_prep_kernel(const FusedPrepParams p) {
    const unsigned long long inst = blockIdx.y;
    const float* Jh = p.Jh + inst * (unsigned long long)(p.L * (p.L - 1));
    const float* Jv = p.Jv + inst * (unsigned long long)((p.L - 1) * p.L);
    const float* hh = p.h ? p.h + inst * (unsigned long long)(p.L * p.L) : nullptr;
    const long idx = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx < p.n_gates) p.gate_m[inst * p.n_gates + idx] = -2.f * Jv[p.gate_jv[idx]];
    if (idx < (long)p.n_tables * 128) {
        const int t = (int)(idx >> 7), var = (int)(idx >> 6) & 1, j = (int)idx & 63;
        const FusedTable tb = p.tables[t];
        float acc = 0.f;
        for (int q = tb.term_begin; q < tb.term_end; ++q) {
            const TableTerm tt = p.terms[q];
            const int ba = tt.posA == 6 ? var : (j >> tt.posA) & 1;
            if (tt.type == OP_DH) {
                const float hv = hh ? hh[tt.row * p.L + tt.col] : 0.f;
                acc += ba ? -hv : hv;
            } else {
                const int bb = tt.posB == 6 ? var : (j >> tt.posB) & 1;
                const float Jc = Jh[tt.row * (p.L - 1) + tt.col];
                acc += (ba == bb) ? Jc : -Jc;
            }
        }
        p.table_out[(inst * p.n_tables + t) * 128 + var * 64 + j] = acc;
    }
}

}  // namespace ttn
