// ttn_fused.cuh -- fused register-phase pass kernel for the Ising Tropical<f32> sweep ("v2").
//
// One launch = one HBM pass.  Each WARP owns a tile of 2^12 state elements,
// 128 per thread, and runs the pass's micro-op program (planner.h, FusedPlan) on it with no
// CTA-level cooperation:
//   * max-plus gates (A2) PAPER.md:242 on a register digit:  v[j] = max(v[j], v[j ^ bit] + m),
//     m = -2 J, the common +J deferred to a scalar (ttn_api.cu): 1 FMNMX + 1/2 FADD2 per element;
//   * diagonal gates (A3), (A4) PAPER.md:247-252 as 128-entry tables in shared memory:
//     v[j] += T[j]  (1/2 FADD2 + 1/4 LDS.128 per element);
//   * layout exchanges A <-> B through the warp's private shared-memory region with 128-bit,
//     bank-conflict-free accesses, synchronised with __syncwarp only.
// Global traffic goes straight between HBM and registers: the LOW tile (columns 0..11) moves
// 128-byte lines; HIGH tiles (columns a..a+8 plus the riding columns 0..2 on the low lane bits)
// move whole 32-byte sectors, four per request.  The kernel is persistent (one CTA per SM);
// programs, gate constants and tables are staged in shared memory once per launch.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>
#include "planner.h"

namespace ttn {

// Warps per CTA (one CTA per SM) and table budget per pass.  The LOW kernel's global accesses
// need no address registers, so it fits 12 warps of 168 registers (3 per scheduler: 87 % of the
// FMNMX peak in the gate phases vs 78 % with 2); the HIGH kernel keeps 8 warps of 255 registers
// so that all 128 strided loads of a tile stay in flight.
constexpr int FWARPS_LOW = 12, FWARPS_HIGH = 8;
constexpr int FMAX_TABLES_LOW = 24, FMAX_TABLES_HIGH = 32;   // 1 KiB each: 2 variants x 128
constexpr int FREGION_F4 = 33 * 32;       // float4 per warp exchange region (low tile: padded rows)
constexpr int FMAX_MOPS = 256;            // micro-ops per pass
__host__ __device__ constexpr int fwarps(bool low) { return low ? FWARPS_LOW : FWARPS_HIGH; }
__host__ __device__ constexpr int fmax_tables(bool low) { return low ? FMAX_TABLES_LOW : FMAX_TABLES_HIGH; }
__host__ __device__ constexpr size_t fsmem_bytes(bool low) {
    return (size_t)fwarps(low) * FREGION_F4 * 16 + (size_t)fmax_tables(low) * 1024 + (size_t)FMAX_MOPS * 8;
}

struct FusedParams {
    int L, a, low, flags, first_layout, last_layout, batch;
    float* state;                       // instance 0
    unsigned long long inst_stride;     // elements between instances
    unsigned long long tiles_per_inst;  // warp tiles (2^12 elements) per instance
    const MicroOp* mops; int n_mops;    // this pass's program
    const float* gate_m; int gate_inst_stride;                    // this pass's slice, instance 0
    const float* tables; int n_tables; unsigned long long table_inst_stride;   // this pass's slice
    float* part_x;                      // [batch][tiles_per_inst] (REDUCE)
};

struct FMop { unsigned ctrl; float m; };  // predecoded: ctrl = code | k << 8 | arg << 16

// (o0, o1) = (a0 + b0, a1 + b1) in one FADD2
__device__ __forceinline__ void add2(float& o0, float& o1, float a0, float a1, float b0, float b1) {
    asm("{ .reg .b64 ra, rb, rc;\n\t"
        "mov.b64 ra, {%2, %3};\n\t"
        "mov.b64 rb, {%4, %5};\n\t"
        "add.f32x2 rc, ra, rb;\n\t"
        "mov.b64 {%0, %1}, rc; }"
        : "=f"(o0), "=f"(o1) : "f"(a0), "f"(a1), "f"(b0), "f"(b1));
}

// ---- gate on register-index bit K: v[j] <- max(v[j], v[j^bit] + m) ---------------------------
template <int K>
__device__ __forceinline__ void fgate(float (&v)[128], const float m) {
    constexpr int B = 1 << K;
    if (K == 0) {
#pragma unroll
        for (int j = 0; j < 128; j += 2) {
            float t0, t1;
            add2(t0, t1, v[j], v[j + 1], m, m);
            v[j] = fmaxf(v[j], t1);
            v[j + 1] = fmaxf(v[j + 1], t0);
        }
    } else {
#pragma unroll
        for (int j = 0; j < 128; j += 2) {
            if ((j & B) == 0) {
                float a0, a1, b0, b1;
                add2(a0, a1, v[j], v[j + 1], m, m);
                add2(b0, b1, v[j + B], v[j + B + 1], m, m);
                v[j] = fmaxf(v[j], b0); v[j + 1] = fmaxf(v[j + 1], b1);
                v[j + B] = fmaxf(v[j + B], a0); v[j + B + 1] = fmaxf(v[j + B + 1], a1);
            }
        }
    }
}

__device__ __forceinline__ void ftable(float (&v)[128], const float4* __restrict__ T) {
#pragma unroll
    for (int q = 0; q < 32; ++q) {
        const float4 t = T[q];
        add2(v[4 * q], v[4 * q + 1], v[4 * q], v[4 * q + 1], t.x, t.y);
        add2(v[4 * q + 2], v[4 * q + 3], v[4 * q + 2], v[4 * q + 3], t.z, t.w);
    }
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

template <bool LOW>
__global__ void __launch_bounds__(fwarps(LOW) * 32, 1) fused_pass_kernel(const FusedParams p) {
    constexpr int FWARPS = fwarps(LOW);
    constexpr int FMAX_TABLES = fmax_tables(LOW);
    extern __shared__ __align__(16) unsigned char fsm_raw[];
    float4* regions = reinterpret_cast<float4*>(fsm_raw);                              // FWARPS * FREGION_F4
    float* s_tab = reinterpret_cast<float*>(fsm_raw + (size_t)FWARPS * FREGION_F4 * 16); // FMAX_TABLES * 256
    FMop* s_mops = reinterpret_cast<FMop*>(fsm_raw + (size_t)FWARPS * FREGION_F4 * 16 + (size_t)FMAX_TABLES * 1024);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    float4* myreg = regions + warp * FREGION_F4;
    const unsigned long long gw = (unsigned long long)blockIdx.x * FWARPS + warp;
    const unsigned long long nw = (unsigned long long)gridDim.x * FWARPS;
    const unsigned long long estride = 1ull << p.a;

    for (int inst = 0; inst < p.batch; ++inst) {
        // ---- stage this instance's program constants and tables (S0 outputs) into shared memory
        __syncthreads();
        for (int i = tid; i < p.n_mops; i += blockDim.x) {
            const MicroOp mo = p.mops[i];
            FMop f;
            f.ctrl = (unsigned)mo.code | ((unsigned)mo.k << 8) | ((unsigned)mo.arg << 16);
            f.m = (mo.code == MC_GATE) ? p.gate_m[(size_t)inst * p.gate_inst_stride + mo.arg] : 0.f;
            s_mops[i] = f;
        }
        {
            const float4* src = reinterpret_cast<const float4*>(p.tables + (size_t)inst * p.table_inst_stride);
            float4* dst = reinterpret_cast<float4*>(s_tab);
            for (int i = tid; i < p.n_tables * 64; i += blockDim.x) dst[i] = src[i];
        }
        __syncthreads();
        float* S = p.state + (unsigned long long)inst * p.inst_stride;

        for (unsigned long long wt = gw; wt < p.tiles_per_inst; wt += nw) {
            // ---- tile geometry ------------------------------------------------------------------
            unsigned long long base;
            int vA = 0, vB = 0;
            if (LOW) {
                base = wt << 12;
                vB = (p.L > F_WLOW) ? (int)(wt & 1ull) : 0;                       // column 12
            } else {
                const int amid = p.a - F_RIDE;
                const unsigned long long tmid = wt & ((1ull << amid) - 1), ttop = wt >> amid;
                base = (tmid << F_RIDE) + (ttop << (p.a + F_WHIGH));
                vA = (int)((base >> (p.a - 1)) & 1ull);                           // column a-1 (>= 3)
                vB = (p.a + F_WHIGH < p.L) ? (int)(ttop & 1ull) : 0;              // column a+9
            }
            float v[128];
            if (p.flags & PASS_INIT) {
#pragma unroll
                for (int j = 0; j < 128; ++j) v[j] = 0.f;                         // tropical one
            } else {
                gmove<LOW, false>(v, S + base, lane, p.first_layout, estride);
            }
            // ---- run the program ------------------------------------------------------------------
            int pc = 0;
            FMop op = s_mops[0];
            for (;;) {
                const unsigned code = op.ctrl & 0xffu;
                if (code == MC_END) break;
                const FMop nxt = s_mops[pc + 1];
                switch (code) {
                    case MC_GATE:
                        switch ((op.ctrl >> 8) & 0xffu) {
                            case 0: fgate<0>(v, op.m); break;
                            case 1: fgate<1>(v, op.m); break;
                            case 2: fgate<2>(v, op.m); break;
                            case 3: fgate<3>(v, op.m); break;
                            case 4: fgate<4>(v, op.m); break;
                            case 5: fgate<5>(v, op.m); break;
                            default: fgate<6>(v, op.m); break;
                        }
                        break;
                    case MC_TABLE: {
                        const int var = ((op.ctrl >> 8) & 0xffu) ? vB : vA;
                        ftable(v, reinterpret_cast<const float4*>(s_tab + ((op.ctrl >> 16) * 2 + var) * 128));
                        break;
                    }
                    case MC_XAB:
                        __syncwarp(); xstore<LOW, 0>(v, myreg, lane); __syncwarp(); xload<LOW, 1>(v, myreg, lane);
                        break;
                    case MC_XBA:
                        __syncwarp(); xstore<LOW, 1>(v, myreg, lane); __syncwarp(); xload<LOW, 0>(v, myreg, lane);
                        break;
                    default: break;
                }
                op = nxt; ++pc;
            }
            // ---- store, or reduce ------------------------------------------------------------------
            if (p.flags & PASS_REDUCE) {
                float mx = v[0];
#pragma unroll
                for (int j = 1; j < 128; ++j) mx = fmaxf(mx, v[j]);
                for (int o = 16; o; o >>= 1) mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, o));
                if (lane == 0) p.part_x[(unsigned long long)inst * p.tiles_per_inst + wt] = mx;
            } else {
                gmove<LOW, true>(v, S + base, lane, p.last_layout, estride);
            }
        }
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
    float* table_out;              // [inst][n_tables][2][128]
};

__global__ void __launch_bounds__(256) fused_prep_kernel(const FusedPrepParams p) {
    const unsigned long long inst = blockIdx.y;
    const float* Jh = p.Jh + inst * (unsigned long long)(p.L * (p.L - 1));
    const float* Jv = p.Jv + inst * (unsigned long long)((p.L - 1) * p.L);
    const float* hh = p.h ? p.h + inst * (unsigned long long)(p.L * p.L) : nullptr;
    const long idx = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx < p.n_gates) p.gate_m[inst * p.n_gates + idx] = -2.f * Jv[p.gate_jv[idx]];
    if (idx < (long)p.n_tables * 256) {
        const int t = (int)(idx >> 8), var = (int)(idx >> 7) & 1, j = (int)idx & 127;
        const FusedTable tb = p.tables[t];
        float acc = 0.f;
        for (int q = tb.term_begin; q < tb.term_end; ++q) {
            const TableTerm tt = p.terms[q];
            const int ba = tt.posA == 7 ? var : (j >> tt.posA) & 1;
            if (tt.type == OP_DH) {
                const float hv = hh ? hh[tt.row * p.L + tt.col] : 0.f;
                acc += ba ? -hv : hv;
            } else {
                const int bb = tt.posB == 7 ? var : (j >> tt.posB) & 1;
                const float Jc = Jh[tt.row * (p.L - 1) + tt.col];
                acc += (ba == bb) ? Jc : -Jc;
            }
        }
        p.table_out[(inst * p.n_tables + t) * 256 + var * 128 + j] = acc;
    }
}

}  // namespace ttn
