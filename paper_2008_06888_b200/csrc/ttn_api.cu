// ttn_api.cu -- the C ABI of include/ttn.h: argument validation, workspace layout, coupling
// upload, kernel launches of one whole sweep, result read-back.  No torch types; no CPU path.
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <map>
#include <mutex>
#include <tuple>
#include <new>
#include <string>
#include <vector>

#include <cuda_runtime.h>

#include "../../include/ttn.h"
#include "planner.h"
#include "ttn_kernels.cuh"
#include "ttn_potts.cuh"
#include "ttn_fused.cuh"
#include "ttn_fcount.cuh"
#include "ttn_chimera.cuh"
#include "ttn_chimera2.cuh"

namespace {

thread_local char g_err[512] = "";

ttn_status fail(ttn_status st, const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof g_err, fmt, ap);
    va_end(ap);
    return st;
}

#define TTN_CUDA(call)                                                                        \
    do {                                                                                      \
        cudaError_t e_ = (call);                                                              \
        if (e_ != cudaSuccess)                                                                \
            return fail(TTN_ECUDA, "%s failed: %s (%s:%d)", #call, cudaGetErrorString(e_),    \
                        __FILE__, __LINE__);                                                  \
    } while (0)

inline size_t align_up(size_t x, size_t a = 256) { return (x + a - 1) / a * a; }

unsigned long long ipow(int q, int e) {
    unsigned long long r = 1;
    for (int i = 0; i < e; ++i) r *= (unsigned long long)q;
    return r;
}

// Test / debug switches (environment TTN_DEBUG_*, honoured only when TTN_ENABLE_DEBUG=1).  They are read ONCE per entry point
// (ttn_workspace_bytes, ttn_plan_describe, ttn_plan_create, the chimera call) into this struct; a
// plan keeps the snapshot it was created with, and no launch path calls getenv.  The tests use them
// to force small tiles, the generic kernels or the fallbacks of the specialised paths.
struct DebugCfg {
    int tmax = -1, ride = -1;     // TTN_DEBUG_TMAX / _RIDE: smaller generic tiles (multi-pass plans on tiny lattices)
    int fused = 1;                // TTN_DEBUG_FUSED=0: generic tile kernels instead of the fused register kernels
    int z2 = 1;                   // TTN_DEBUG_Z2=0: never use the global-flip reduction (h = 0)
    int nobeam = 0, nb = -1;      // Potts: TTN_DEBUG_NOBEAM, TTN_DEBUG_NB (gate-block size)
    int nolowpf = 0, nogroup = 0, nosweep = 0;   // ground_config forward: no LOW prefetch / instance groups / one-launch sweep
    int bt_multi = 0;             // backward pass: one launch pair per row even for batches of small lattices
    int timing = 0;               // per-pass device times on stderr
    int ckpt_k = 0;               // TTN_DEBUG_CKPT_K=k: ground_config keeps a checkpoint every k rows + recompute (any L)
    int nomerge = 0;              // TTN_DEBUG_NOMERGE: ground_config forward with one pass per tile and row (no merged passes)
    int ch_persm = 512, ch_nocell0 = 0;          // chimera: CTAs per SM, generic kernel for the r = 0 cells
};
DebugCfg read_debug() {
    DebugCfg d;
    // opt-in: without TTN_ENABLE_DEBUG=1 (set by tests/conftest.py) no TTN_DEBUG_* variable is looked at, so a
    // stray one in a user's environment cannot change a workspace size or a kernel path
    { const char* en = getenv("TTN_ENABLE_DEBUG"); if (!en || atoi(en) != 1) return d; }
    auto geti = [](const char* name, int& v) { if (const char* e = getenv(name)) v = atoi(e); };
    auto flag = [](const char* name, int& v) { v = getenv(name) != nullptr; };
    geti("TTN_DEBUG_TMAX", d.tmax); geti("TTN_DEBUG_RIDE", d.ride); geti("TTN_DEBUG_FUSED", d.fused);
    geti("TTN_DEBUG_Z2", d.z2); geti("TTN_DEBUG_NB", d.nb); geti("TTN_DEBUG_CH_PERSM", d.ch_persm);
    geti("TTN_DEBUG_CKPT_K", d.ckpt_k);
    flag("TTN_DEBUG_NOBEAM", d.nobeam); flag("TTN_DEBUG_NOLOWPF", d.nolowpf); flag("TTN_DEBUG_NOGROUP", d.nogroup);
    flag("TTN_DEBUG_NOSWEEP", d.nosweep); flag("TTN_DEBUG_BT_MULTI", d.bt_multi); flag("TTN_DEBUG_TIMING", d.timing);
    flag("TTN_DEBUG_CH_NOCELL0", d.ch_nocell0); flag("TTN_DEBUG_NOMERGE", d.nomerge);
    if (d.ch_persm < 1) d.ch_persm = 512;
    return d;
}

// Tile capacity (log_q of elements per CTA tile) and riding digits of the generic path.
struct TileCfg { int Tmax, ride; };
// z3: the Potts CTA holds the three member tiles of a rotation orbit: one digit less per member
TileCfg tile_cfg(int q, bool count, const DebugCfg& dbg, bool z3 = false) {
    TileCfg t;
    if (q == 2) t = count ? TileCfg{13, 3} : TileCfg{14, 3};   // 96 KiB / 64 KiB of smem
    else t = count ? TileCfg{8, 2} : TileCfg{9, 2};           // 3^8*12 = 77 KiB / 3^9*4 = 77 KiB
    if (q == 3 && z3) t.Tmax -= 1;
    // Debug/test override (smaller tiles only): lets tiny lattices exercise multi-pass schedules.
    if (dbg.tmax >= 2 && dbg.tmax <= t.Tmax) t.Tmax = dbg.tmax;
    if (dbg.ride >= 0 && dbg.ride < t.Tmax) t.ride = dbg.ride;
    if (t.ride >= t.Tmax) t.ride = t.Tmax - 1;
    return t;
}

bool limits_ok(int q, int L, bool count, bool config) {
    if (L < 1) return false;
    if (q == 2) {
        if (config) return L <= 32;
        return count ? L <= 32 : L <= 34;
    }
    if (q == 3) return !config && L <= 20;
    return false;
}

// Checkpoints of ttn_ground_config ("checkpointing").  k = 0: every row boundary C_r has
// its own buffer (L buffers).  k > 1 (L > 28, where L buffers no longer fit): C_r is kept for
// r = 0, k, 2k, ... and r = L-1 only; the backward pass re-sweeps each segment (a, b) of rows between
// two kept checkpoints from C_a into a ring of k - 1 scratch buffers, backtracks through it, and moves
// on to the segment below: n_stored + k - 1 buffers, k ~ sqrt(L), and one extra forward sweep in total.
struct CkptScheme {
    int L = 0, k = 0, n_stored = 0, n_buf = 0;
    bool stored(int r) const { return k == 0 || r % k == 0 || r == L - 1; }
    int stored_slot(int r) const { return k == 0 ? r : (r % k == 0 ? r / k : n_stored - 1); }
    int prev_stored(int b) const { return k == 0 ? b - 1 : ((b - 1) / k) * k; }   // largest stored row < b
    int ring_slot(int a, int r) const { return n_stored + (r - a - 1); }           // a < r < next stored row
};
CkptScheme ckpt_scheme(int L, bool fused, const DebugCfg& dbg) {
    CkptScheme c; c.L = L; c.k = 0; c.n_stored = L; c.n_buf = L;
    int k = 0;
    if (fused && dbg.ckpt_k > 1) k = dbg.ckpt_k;
    else if (fused && L > 28) { k = 1; while (k * k < L) ++k; }
    if (k <= 1 || k >= L - 1) return c;
    c.k = k; c.n_stored = 0;
    for (int r = 0; r < L; ++r) if (r % k == 0 || r == L - 1) ++c.n_stored;
    c.n_buf = c.n_stored + k - 1;
    return c;
}

struct Layout {
    size_t x = 0, n = 0, ckpt = 0, Jh = 0, Jv = 0, h = 0, ops = 0, part_x = 0, part_n = 0,
           amax_v = 0, amax_s = 0, out_x = 0, out_n = 0, out_s = 0, sigma = 0, total = 0;
    size_t f_mops = 0, f_gate_rc = 0, f_gate_k = 0, f_final = 0, g_gate_k = 0, g_fin = 0, f_sweep = 0;
    unsigned long long NS = 0, max_tiles = 0;
    int amax_blocks = 0;
    int f_max_gates = 0, f_max_mops = 0;
    CkptScheme ck;
};

// The fused register-phase paths: Ising Tropical<f32> energy for L >= 12 (ttn_fused.cuh) and Ising
// CountingTropical<f32,f64> for L >= 10 (ttn_fcount.cuh).
bool i16_eligible(int q, int L, const DebugCfg& dbg) {
    return dbg.fused != 0 && q == 2 && L >= ttn::GEOM_I16.WLOW;
}
bool fused_eligible(int q, int L, bool count, bool config, const DebugCfg& dbg) {
    if (dbg.fused == 0 || q != 2) return false;
    return count ? L >= ttn::CW_LOW : L >= ttn::F_WLOW;      // config: row-aligned f32 plan
}
// Colour-rotation (Z3) reduction of the Potts sweeps (planner.h): always valid (no fields); used when the
// reduced state of L - 1 digits spans more than one member tile, so that every rotation orbit has three tiles.
bool z3_eligible(int q, int L, bool count, const DebugCfg& dbg) {
    if (q != 3 || dbg.z2 == 0 || L < 3) return false;
    return L - 1 > tile_cfg(3, count, dbg, true).Tmax;
}

// Global-flip (Z2) reduction (planner.h): h = 0 only; the half-state must span at least two LOW tiles
// (a tile and its complement).  Geometry of the call, or nullptr.
const ttn::FusedGeom* z2_geom(int q, int L, ttn_call call, bool has_field, const DebugCfg& dbg) {
    if (dbg.fused == 0 || dbg.z2 == 0 || q != 2 || has_field) return nullptr;
    if ((call == TTN_CALL_ENERGY || call == TTN_CALL_ENERGY_Z2 || call == TTN_CALL_CONFIG || call == TTN_CALL_CONFIG_Z2) &&
        L >= ttn::GEOM_F32_Z2.WLOW + 1) return &ttn::GEOM_F32_Z2;
    if ((call == TTN_CALL_COUNT || call == TTN_CALL_COUNT_Z2) && L >= ttn::GEOM_COUNT_Z2.WLOW + 1) return &ttn::GEOM_COUNT_Z2;
    if ((call == TTN_CALL_ENERGY_I16 || call == TTN_CALL_ENERGY_I16_Z2) && L >= ttn::GEOM_I16_Z2.WLOW + 1) return &ttn::GEOM_I16_Z2;
    return nullptr;
}

// The op list of a plan holds the L(L-1) gates of the sweep (diagonal frame: no diagonal op).
// z2: the stored state is the half with column 0 up: q^(L-1) elements (every size below follows NS)
Layout make_layout(int q, int L, bool count, bool config, int batch, const DebugCfg& dbg, bool i16 = false, bool z2 = false) {
    Layout y;
    y.NS = ipow(q, z2 ? L - 1 : L);
    const TileCfg tc = tile_cfg(q, count, dbg, q == 3 && z2);
    // every pass of a plan stages tiles of q^min(L, Tmax) elements
    y.max_tiles = y.NS / ipow(q, tc.Tmax < L ? tc.Tmax : L);     // (Z3: three tiles per partial: an upper bound)
    if (fused_eligible(q, L, count, config, dbg) && y.max_tiles < 1024) y.max_tiles = 1024;   // one partial per CTA
    if (y.max_tiles == 0) y.max_tiles = 1;
    size_t off = 0;
    auto take = [&](size_t bytes) { size_t o = off; off = align_up(off + bytes); return o; };
    y.x = take((size_t)batch * y.NS * (i16 ? 2 : 4));
    if (count) y.n = take((size_t)batch * y.NS * 8);
    y.ck = ckpt_scheme(L, config && fused_eligible(q, L, count, config, dbg), dbg);
    if (config) y.ckpt = take((size_t)batch * y.ck.n_buf * y.NS * 4);
    y.Jh = take((size_t)batch * L * (L - 1) * 4 + 4);
    y.Jv = take((size_t)batch * (L - 1) * L * 4 + 4);
    y.h = take((size_t)batch * L * L * 4);
    y.ops = take((size_t)(L * L + 8) * sizeof(ttn::Op));
    y.g_gate_k = take((size_t)batch * (L * L + 8) * 8 * 4);
    y.g_fin = take((size_t)batch * 2 * ttn::GMAX_L * 4);
    y.part_x = take((size_t)batch * y.max_tiles * 4);
    y.part_n = take((size_t)batch * y.max_tiles * 8);
    unsigned long long nb = (y.NS + 256ull * 16 - 1) / (256ull * 16);
    y.amax_blocks = (int)(nb < 1 ? 1 : (nb > 1024 ? 1024 : nb));
    y.amax_v = take((size_t)batch * y.amax_blocks * 4);
    y.amax_s = take((size_t)batch * y.amax_blocks * 8);
    y.out_x = take((size_t)batch * 4);
    y.out_n = take((size_t)batch * 8);
    y.out_s = take((size_t)batch * 8);
    y.sigma = take((size_t)batch * L * L);
    if (fused_eligible(q, L, count, config, dbg)) {
        y.f_max_gates = L * L; y.f_max_mops = 4 * L * L + 64;
        y.f_mops = take((size_t)y.f_max_mops * sizeof(ttn::MicroOp));
        y.f_gate_rc = take((size_t)y.f_max_gates * 4);
        y.f_gate_k = take((size_t)batch * y.f_max_gates * 8 * 4);
        y.f_final = take((size_t)batch * ttn::FFINAL_FLOATS * 4);
        y.f_sweep = take((size_t)(4 * L + 8) * sizeof(ttn::FusedParams));     // fused_sweep_kernel: one entry per pass
    }
    y.total = off;
    return y;
}

template <typename K>
ttn_status set_smem(K kernel, size_t bytes) {
    TTN_CUDA(cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes));
    return TTN_OK;
}

}  // namespace

struct ttn_plan {
    int q, L, batch;
    ttn_call call;
    bool count, config, has_field;
    ttn::Plan plan;
    ttn::FusedPlan fplan;
    bool fused = false, i16 = false;
    bool merged = false;           // row plan with merged passes (MC_CKPT): runs on fused_sweep_kernel only
    bool z2 = false;               // global-flip reduction: the state is the half with column 0 up (h = 0)
    DebugCfg dbg;                  // the debug switches as they were when the plan was created
    int fused_grid = 0;
    int sms = 0;
    // row-aligned (config) fused plans: passes of row r = [row_pass[r], row_pass[r + 1]); buffer slot that
    // holds C_r at the moment (-1: none -- the row's result lives in the in-place state V)
    std::vector<int> row_pass, slot_of_row;
    int sweep_grid = 0;             // > 0: fused_sweep_kernel runs every pass in one launch (table at lay.f_sweep)
    std::vector<ttn::FusedParams> sweep_params;
    Layout lay;
    unsigned char* ws;
    std::vector<double> defer;     // per instance: sum of the +J constants factored out of the gates
    int launches;
};

static ttn::Plan plan_for(int q, int L, ttn_call call, bool has_field, const DebugCfg& dbg) {
    const bool count = (call == TTN_CALL_COUNT);
    if (z3_eligible(q, L, count, dbg)) {              // Potts on the colour-rotation-reduced state: L - 1 digits + column 0
        const TileCfg tc = tile_cfg(q, count, dbg, true);
        const int Ld = L - 1;
        ttn::Plan p = ttn::make_plan(q, Ld, false, false, tc.Tmax, tc.ride, /*vcol=*/true);
        if (!dbg.nobeam) {
            static std::map<std::tuple<int, int, int>, ttn::Plan> zcache;      // memo, as below
            static std::mutex zmu;
            std::lock_guard<std::mutex> lock(zmu);
            const auto key = std::make_tuple(Ld, tc.Tmax, tc.ride);
            auto it = zcache.find(key);
            if (it == zcache.end()) it = zcache.emplace(key, ttn::make_plan_beam(q, Ld, tc.Tmax, tc.ride, 256, true)).first;
            if (!it->second.passes.empty() && it->second.passes.size() < p.passes.size()) p = it->second;
        }
        int max_nb = count ? ttn::POTTS_MAX_NB_COUNT : 3;
        if (dbg.nb >= 1 && dbg.nb <= max_nb) max_nb = dbg.nb;
        ttn::mark_gate_blocks(p, max_nb);
        return p;
    }
    const TileCfg tc = tile_cfg(q, count, dbg);
    ttn::Plan p = ttn::make_plan(q, L, has_field, call == TTN_CALL_CONFIG, tc.Tmax, tc.ride);
    if (q == 3 && L > tc.Tmax && !dbg.nobeam) {       // multi-pass Potts sweep: search the tile order
        // The one piece of process-wide state in the library: a memo of beam-searched Potts schedules
        // (a pure function of (L, Tmax, ride), ~1 s to compute at L = 18), guarded by a mutex.
        static std::map<std::tuple<int, int, int>, ttn::Plan> cache;
        static std::mutex mu;
        std::lock_guard<std::mutex> lock(mu);
        const auto key = std::make_tuple(L, tc.Tmax, tc.ride);
        auto it = cache.find(key);
        if (it == cache.end()) it = cache.emplace(key, ttn::make_plan_beam(q, L, tc.Tmax, tc.ride)).first;
        if (!it->second.passes.empty() && it->second.passes.size() < p.passes.size()) p = it->second;
    }
    if (q == 3) {
        int max_nb = count ? ttn::POTTS_MAX_NB_COUNT : 3;
        if (dbg.nb >= 1 && dbg.nb <= max_nb) max_nb = dbg.nb;
        ttn::mark_gate_blocks(p, max_nb);
    }
    return p;
}

template <int Q, bool COUNT>
static ttn_status launch_pass(const ttn_plan* P, const ttn::Pass& ps, cudaStream_t st) {
    const Layout& y = P->lay;
    ttn::PassParams pp{};
    const bool z3 = Q == 3 && P->z2;           // (the plan's "reduced by the symmetry" flag)
    pp.z3 = z3 ? 1 : 0;
    pp.L = z3 ? P->L - 1 : P->L; pp.lo = ps.lo; pp.a = ps.a; pp.b = ps.b; pp.T = ps.lo + (ps.b - ps.a);
    pp.P_lo = ipow(Q, ps.lo); pp.P_a = ipow(Q, ps.a); pp.P_mid = ipow(Q, ps.a - ps.lo); pp.P_b = ipow(Q, ps.b);
    pp.n_tile = (unsigned)ipow(Q, pp.T);
    pp.tiles_per_inst = y.NS / pp.n_tile;
    float* V = reinterpret_cast<float*>(P->ws + y.x);
    float* CK = reinterpret_cast<float*>(P->ws + y.ckpt);
    auto buf = [&](int id, unsigned long long& stride) -> float* {
        if (id < 0) { stride = y.NS; return V; }
        stride = (unsigned long long)y.ck.n_buf * y.NS;
        return CK + (unsigned long long)id * y.NS;
    };
    pp.src_x = buf(ps.src_buf, pp.src_stride);
    pp.dst_x = buf(ps.dst_buf, pp.dst_stride);
    pp.src_n = pp.dst_n = COUNT ? reinterpret_cast<double*>(P->ws + y.n) : nullptr;
    pp.ops = reinterpret_cast<const ttn::Op*>(P->ws + y.ops) + ps.op_begin;
    pp.n_ops = ps.op_end - ps.op_begin;
    pp.gate_k = reinterpret_cast<const float*>(P->ws + y.g_gate_k) + (size_t)ps.op_begin * 8;
    pp.gate_inst_stride = (unsigned long long)P->plan.ops.size() * 8;
    pp.fin = reinterpret_cast<const float*>(P->ws + y.g_fin);
    pp.flags = ps.flags;
    pp.part_x = reinterpret_cast<float*>(P->ws + y.part_x);
    pp.part_n = reinterpret_cast<double*>(P->ws + y.part_n);
    const size_t smem = (size_t)pp.n_tile * (COUNT ? 12 : 4);
    // Z3: a work unit is a rotation orbit of three tiles
    const unsigned long long units_per_inst = z3 ? pp.tiles_per_inst / 3 : pp.tiles_per_inst;
    const unsigned long long grid = units_per_inst * (unsigned long long)P->batch;
    if (grid > 0x7fffffffull) return fail(TTN_EUNSUPPORTED, "grid too large");
    if constexpr (Q == 3) {    // Potts: register-blocked gates (ttn_potts.cuh)
        // persistent CTAs, two residents per SM (ttn_potts.cuh)
        if (pp.n_ops > ttn::POTTS_MAX_OPS) return fail(TTN_EUNSUPPORTED, "too many gates in one Potts pass");
        if (pp.T > 9) return fail(TTN_EUNSUPPORTED, "Potts tiles hold at most 3^9 elements");
        const int sms = P->sms;                         // of the device the plan was created on
        const unsigned ctas = grid < 2ull * sms ? (unsigned)grid : 2u * (unsigned)sms;
        const size_t psmem = z3 ? ttn::potts_z3_bytes(pp.n_tile, COUNT) : ttn::potts_buf_bytes(pp.n_tile, COUNT);
        ttn_status s = TTN_OK;
        if (pp.n_tile * (z3 ? 3u : 1u) / 27 <= 128) {                  // tiny lattices
            s = set_smem(ttn::potts_pass_kernel<COUNT, 128>, psmem);
            if (s != TTN_OK) return s;
            ttn::potts_pass_kernel<COUNT, 128><<<ctas, 128, psmem, st>>>(pp, (unsigned)grid);
        } else {
            constexpr int TH = COUNT ? ttn::POTTS_THREADS_COUNT : ttn::POTTS_THREADS;
            s = set_smem(ttn::potts_pass_kernel<COUNT, TH>, psmem);
            if (s != TTN_OK) return s;
            ttn::potts_pass_kernel<COUNT, TH><<<ctas, TH, psmem, st>>>(pp, (unsigned)grid);
        }
    } else {
        ttn_status s = set_smem(ttn::pass_kernel<Q, COUNT>, smem);
        if (s != TTN_OK) return s;
        unsigned threads = pp.n_tile / Q >= 512 ? 512 : (pp.n_tile / Q < 32 ? 32 : ((pp.n_tile / Q + 31) / 32 * 32));
        ttn::pass_kernel<Q, COUNT><<<(unsigned)grid, threads, smem, st>>>(pp);
    }
    TTN_CUDA(cudaGetLastError());
    if (ps.flags & ttn::PASS_REDUCE) {
        ttn::final_reduce_kernel<COUNT><<<P->batch, 256, 0, st>>>(
            pp.part_x, pp.part_n, units_per_inst, reinterpret_cast<float*>(P->ws + y.out_x),
            reinterpret_cast<double*>(P->ws + y.out_n));
        TTN_CUDA(cudaGetLastError());
    }
    return TTN_OK;
}

// out_pp != NULL: only fill the parameters (force_group instances per CTA at a time) and the grid.
static ttn_status launch_fused_pass(const ttn_plan* P, const ttn::FusedPass& ps, cudaStream_t st,
                                    ttn::FusedParams* out_pp = nullptr, int force_group = 0, unsigned* out_grid = nullptr);
static ttn_status launch_fused_pass(const ttn_plan* P, const ttn::FusedPass& ps, cudaStream_t st,
                                    ttn::FusedParams* out_pp, int force_group, unsigned* out_grid) {
    const Layout& y = P->lay;
    const ttn::FusedPlan& fp = P->fplan;
    ttn::FusedParams pp{};
    pp.L = P->L; pp.a = ps.a; pp.low = ps.low; pp.flags = ps.flags; pp.batch = P->batch;
    pp.first_layout = ps.first_layout; pp.last_layout = ps.last_layout;
    pp.state = reinterpret_cast<float*>(P->ws + y.x);
    pp.inst_stride = y.NS;
    pp.tiles_per_inst = y.NS >> 12;
    pp.src = pp.state; pp.src_stride = pp.inst_stride;
    if (P->config) {           // row-aligned plan: checkpoints C_r = V''_r, [inst][L][2^L]
        float* CK = reinterpret_cast<float*>(P->ws + y.ckpt);
        const unsigned long long cstride = (unsigned long long)y.ck.n_buf * y.NS;
        const int ss = ps.src_buf >= 0 ? P->slot_of_row[ps.src_buf] : -1, ds = ps.dst_buf >= 0 ? P->slot_of_row[ps.dst_buf] : -1;
        if (ss >= 0) { pp.src = CK + (unsigned long long)ss * y.NS; pp.src_stride = cstride; }
        if (ds >= 0) { pp.state = CK + (unsigned long long)ds * y.NS; pp.inst_stride = cstride; }
        if (ps.ckpt_buf >= 0) { pp.ckpt = CK + (unsigned long long)P->slot_of_row[ps.ckpt_buf] * y.NS; pp.ckpt_stride = cstride; }
    }
    pp.L_cols = P->L;
    if (P->i16) {           // the kernel sees the lattice of 32-bit words: column c >= 1 = word digit c - 1
        const int off = P->z2 ? 2 : 1;     // (flip-reduced: the half-state's column 1 is the half of a word)
        pp.L = P->L - off; pp.a = ps.low ? 0 : ps.a - off;
        pp.L_cols = P->L - (off - 1);      // digits of the element index
        pp.inst_stride = y.NS >> 1; pp.tiles_per_inst = y.NS >> 13;
        pp.src = pp.state; pp.src_stride = pp.inst_stride;
    } else if (P->z2) {     // the kernel sees the half-state over columns 1 .. L-1: column c = digit c - 1
        pp.L = P->L - 1; pp.a = ps.low ? 0 : ps.a - 1;
    }
    const int a_mem = pp.a;
    pp.mops = reinterpret_cast<const ttn::MicroOp*>(P->ws + y.f_mops) + ps.mop_begin;
    pp.n_mops = ps.mop_end - ps.mop_begin;
    pp.gate_k = reinterpret_cast<const float*>(P->ws + y.f_gate_k) + (size_t)ps.gate_begin * 8;
    pp.n_gates = ps.gate_end - ps.gate_begin;
    pp.gate_inst_stride = (unsigned long long)fp.gate_rc.size() * 8;
    pp.final_tab = reinterpret_cast<const float*>(P->ws + y.f_final);
    pp.part_x = reinterpret_cast<float*>(P->ws + y.part_x);
    pp.stride_bytes = 4u << a_mem;    // a <= L - 9 <= 25
    pp.prefetch_pc = 0;
    for (int k = ps.mop_begin; k < ps.mop_end; ++k)
        if (fp.mops[k].code == ttn::MC_XAB || fp.mops[k].code == ttn::MC_XBA) pp.prefetch_pc = k - ps.mop_begin + 1;
    if (a_mem > 18) pp.prefetch_pc = -1;     // > 256 distinct 2 MiB pages per tile: synchronous loads
    unsigned long long grid = (unsigned long long)P->fused_grid;
    const int nw = ttn::fwarps(ps.low != 0, P->i16 ? 1 : 0);
    // batches of small lattices: one CTA per instance at a time instead of the whole grid per instance
    pp.cta_per_inst = (P->batch > 1 && pp.tiles_per_inst < (unsigned long long)nw * grid) ? 1 : 0;
    if (pp.cta_per_inst) {
        if (grid > (unsigned long long)P->batch) grid = (unsigned long long)P->batch;
    } else {
        const unsigned long long need = (pp.tiles_per_inst + nw - 1) / nw;
        if (grid > need) grid = need;
    }
    pp.part_stride = pp.cta_per_inst ? 1 : (int)grid;
    if (ps.low && P->dbg.nolowpf) pp.prefetch_pc = -1;
    pp.igroup = 1;
    { int sh = 0; while ((1ull << sh) < pp.tiles_per_inst) ++sh; pp.tpi_shift = sh; }
    if (pp.cta_per_inst && !P->i16 && !P->z2 && !(ps.flags & ttn::PASS_REDUCE) && !P->dbg.nogroup) {
        // instances per CTA at a time: fewest rounds of the 12 warps (HIGH: of the 3 warp groups) over
        // the flat tile list of K instances, times the rounds of CTA groups over the grid
        const unsigned long long tpi = pp.tiles_per_inst, slots = ps.low ? (unsigned long long)nw : (unsigned long long)(nw / 4);
        const unsigned long long unit = ps.low ? 1 : 4;
        double best = 0; int bestK = 1;
        for (int K = 1; K <= 8; ++K) {
            if ((size_t)K * (pp.n_gates * 2 + 2) > (size_t)(ttn::FMAX_GATES + 1) * 2) break;
            const unsigned long long groups = ((unsigned long long)P->batch + K - 1) / K;
            const unsigned long long waves = (groups + P->fused_grid - 1) / P->fused_grid;
            const unsigned long long rounds = ((K * tpi + unit - 1) / unit + slots - 1) / slots;
            const double cost = (double)(waves * rounds);
            if (K == 1 || cost < best) { best = cost; bestK = K; }
        }
        pp.igroup = force_group > 0 ? force_group : bestK;
    }
    if (out_pp) {
        if (!pp.cta_per_inst || (ps.flags & ttn::PASS_REDUCE) || P->i16) return fail(TTN_EUNSUPPORTED, "pass not eligible for the one-launch sweep");
        if ((size_t)pp.igroup * (pp.n_gates * 2 + 2) > (size_t)(ttn::FMAX_GATES + 1) * 2) return fail(TTN_EUNSUPPORTED, "instance group too large");
        const unsigned long long groups = ((unsigned long long)P->batch + pp.igroup - 1) / pp.igroup;
        if (out_grid) *out_grid = (unsigned)(groups < (unsigned long long)P->fused_grid ? groups : (unsigned long long)P->fused_grid);
        *out_pp = pp;
        return TTN_OK;
    }
    if (pp.igroup > 1) {
        const unsigned long long groups = ((unsigned long long)P->batch + pp.igroup - 1) / pp.igroup;
        grid = groups < (unsigned long long)P->fused_grid ? groups : (unsigned long long)P->fused_grid;
        if (ps.low) ttn::fused_pass_kernel<true, 0, true><<<(unsigned)grid, nw * 32, ttn::fsmem_bytes(true), st>>>(pp);
        else ttn::fused_pass_kernel<false, 0, true><<<(unsigned)grid, nw * 32, ttn::fsmem_bytes(false), st>>>(pp);
    } else {
        const bool red = (ps.flags & ttn::PASS_REDUCE) != 0;
#define TTN_FUSED_LAUNCH(LOW_, ELEM_, RED_)                                                                             \
        ttn::fused_pass_kernel<LOW_, ELEM_, false, RED_><<<(unsigned)grid, nw * 32, ttn::fsmem_bytes(LOW_, ELEM_), st>>>(pp)
        if (P->i16 && P->z2 && ps.low) {
            if (red) ttn::fused_pass_kernel<true, 1, false, true, true><<<(unsigned)grid, nw * 32, ttn::fsmem_bytes(true, 1), st>>>(pp);
            else ttn::fused_pass_kernel<true, 1, false, false, true><<<(unsigned)grid, nw * 32, ttn::fsmem_bytes(true, 1), st>>>(pp);
        } else if (P->i16) {
            if (ps.low) { if (red) TTN_FUSED_LAUNCH(true, 1, true); else TTN_FUSED_LAUNCH(true, 1, false); }
            else { if (red) TTN_FUSED_LAUNCH(false, 1, true); else TTN_FUSED_LAUNCH(false, 1, false); }
        } else if (P->z2 && ps.low) {      // warp pairs on complementary tiles, flip gates
            if (red) ttn::fused_pass_kernel<true, 0, false, true, true><<<(unsigned)grid, nw * 32, ttn::fsmem_bytes(true), st>>>(pp);
            else ttn::fused_pass_kernel<true, 0, false, false, true><<<(unsigned)grid, nw * 32, ttn::fsmem_bytes(true), st>>>(pp);
        } else {
            if (ps.low) { if (red) TTN_FUSED_LAUNCH(true, 0, true); else TTN_FUSED_LAUNCH(true, 0, false); }
            else { if (red) TTN_FUSED_LAUNCH(false, 0, true); else TTN_FUSED_LAUNCH(false, 0, false); }
        }
#undef TTN_FUSED_LAUNCH
    }
    TTN_CUDA(cudaGetLastError());
    if (ps.flags & ttn::PASS_REDUCE) {
        // one partial per CTA and instance
        ttn::final_reduce_kernel<false><<<P->batch, 256, 0, st>>>(
            pp.part_x, nullptr, (unsigned long long)pp.part_stride, reinterpret_cast<float*>(P->ws + y.out_x), nullptr);
        TTN_CUDA(cudaGetLastError());
    }
    return TTN_OK;
}

static ttn_status launch_fcount_pass(const ttn_plan* P, const ttn::FusedPass& ps, cudaStream_t st) {
    const Layout& y = P->lay;
    const ttn::FusedPlan& fp = P->fplan;
    ttn::CountParams cp{};
    ttn::FusedParams& pp = cp.f;
    pp.L = P->L; pp.a = ps.a; pp.low = ps.low; pp.flags = ps.flags; pp.batch = P->batch;
    if (P->z2) { pp.L = P->L - 1; pp.a = ps.low ? 0 : ps.a - 1; }      // half-state: column c = digit c - 1
    pp.first_layout = ps.first_layout; pp.last_layout = ps.last_layout;
    pp.state = reinterpret_cast<float*>(P->ws + y.x);
    cp.state_n = reinterpret_cast<double*>(P->ws + y.n);
    pp.inst_stride = y.NS;
    pp.src = pp.state; pp.src_stride = y.NS;
    pp.tiles_per_inst = y.NS >> 10;
    pp.mops = reinterpret_cast<const ttn::MicroOp*>(P->ws + y.f_mops) + ps.mop_begin;
    pp.n_mops = ps.mop_end - ps.mop_begin;
    pp.gate_k = reinterpret_cast<const float*>(P->ws + y.f_gate_k) + (size_t)ps.gate_begin * 8;
    pp.n_gates = ps.gate_end - ps.gate_begin;
    pp.gate_inst_stride = (unsigned long long)fp.gate_rc.size() * 8;
    pp.final_tab = reinterpret_cast<const float*>(P->ws + y.f_final);
    pp.part_x = reinterpret_cast<float*>(P->ws + y.part_x);
    cp.part_n = reinterpret_cast<double*>(P->ws + y.part_n);
    pp.stride_bytes = 4u << pp.a;
    pp.prefetch_pc = -1;
    unsigned long long grid = (unsigned long long)P->fused_grid;
    const int nw = ttn::CWARPS;
    pp.cta_per_inst = (P->batch > 1 && pp.tiles_per_inst < (unsigned long long)nw * grid) ? 1 : 0;
    if (pp.cta_per_inst) {
        if (grid > (unsigned long long)P->batch) grid = (unsigned long long)P->batch;
    } else {
        const unsigned long long need = (pp.tiles_per_inst + nw - 1) / nw;
        if (grid > need) grid = need;
    }
    pp.part_stride = pp.cta_per_inst ? 1 : (int)grid;
    if (ps.low && P->z2) ttn::fcount_pass_kernel<true, true><<<(unsigned)grid, nw * 32, ttn::csmem_bytes(), st>>>(cp);
    else if (ps.low) ttn::fcount_pass_kernel<true><<<(unsigned)grid, nw * 32, ttn::csmem_bytes(), st>>>(cp);
    else ttn::fcount_pass_kernel<false><<<(unsigned)grid, nw * 32, ttn::csmem_bytes(), st>>>(cp);
    TTN_CUDA(cudaGetLastError());
    if (ps.flags & ttn::PASS_REDUCE) {
        ttn::final_reduce_kernel<true><<<P->batch, 256, 0, st>>>(
            pp.part_x, cp.part_n, (unsigned long long)pp.part_stride, reinterpret_cast<float*>(P->ws + y.out_x),
            reinterpret_cast<double*>(P->ws + y.out_n));
        TTN_CUDA(cudaGetLastError());
    }
    return TTN_OK;
}

static ttn_status setup_fcount(ttn_plan* P, cudaStream_t st) {
    const Layout& y = P->lay;
    ttn::FusedPlan& fp = P->fplan;
    if ((int)fp.gate_rc.size() > y.f_max_gates || (int)fp.mops.size() > y.f_max_mops)
        return fail(TTN_EUNSUPPORTED, "fused plan exceeds its workspace bounds");
    for (const auto& ps : fp.passes)
        if (ps.mop_end - ps.mop_begin > ttn::FMAX_MOPS || ps.gate_end - ps.gate_begin > ttn::FMAX_GATES ||
            (ps.low && (ps.first_layout != 1 || ps.last_layout != 1)))
            return fail(TTN_EUNSUPPORTED, "fused pass program out of bounds");
    TTN_CUDA(cudaMemcpyAsync(P->ws + y.f_mops, fp.mops.data(), fp.mops.size() * sizeof(ttn::MicroOp), cudaMemcpyHostToDevice, st));
    TTN_CUDA(cudaMemcpyAsync(P->ws + y.f_gate_rc, fp.gate_rc.data(), fp.gate_rc.size() * 4, cudaMemcpyHostToDevice, st));
    ttn::CountPrepParams q{};
    q.L = P->L; q.n_gates = (int)fp.gate_rc.size();
    q.gate_rc = reinterpret_cast<const int*>(P->ws + y.f_gate_rc);
    q.Jh = reinterpret_cast<const float*>(P->ws + y.Jh);
    q.Jv = reinterpret_cast<const float*>(P->ws + y.Jv);
    q.h = P->has_field ? reinterpret_cast<const float*>(P->ws + y.h) : nullptr;
    q.gate_k = reinterpret_cast<float*>(P->ws + y.f_gate_k);
    q.final_tab = reinterpret_cast<float*>(P->ws + y.f_final);
    const ttn::FusedPass& lastp = fp.passes.back();
    q.fin_low = lastp.low; q.fin_layout = lastp.last_layout; q.fin_a = lastp.a;
    if (P->z2) q.fin_a = lastp.low ? 0 : lastp.a - 1;
    q.col_off = P->z2 ? 1 : 0;
    long work = ttn::CFINAL_FLOATS; if (q.n_gates > work) work = q.n_gates;
    dim3 grid((unsigned)((work + 255) / 256), (unsigned)P->batch);
    ttn::fcount_prep_kernel<<<grid, 256, 0, st>>>(q);
    TTN_CUDA(cudaGetLastError());
    TTN_CUDA(cudaFuncSetAttribute(ttn::fcount_pass_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ttn::csmem_bytes()));
    TTN_CUDA(cudaFuncSetAttribute(ttn::fcount_pass_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ttn::csmem_bytes()));
    TTN_CUDA(cudaFuncSetAttribute(ttn::fcount_pass_kernel<true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ttn::csmem_bytes()));
    int dev = 0, sms = 0;
    TTN_CUDA(cudaGetDevice(&dev));
    TTN_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    P->fused_grid = sms;
    return TTN_OK;
}

// Uploads the fused program and runs the S0 prep kernel (gate constants + final table).
static ttn_status setup_fused(ttn_plan* P, cudaStream_t st) {
    const Layout& y = P->lay;
    ttn::FusedPlan& fp = P->fplan;
    if ((int)fp.gate_rc.size() > y.f_max_gates || (int)fp.mops.size() > y.f_max_mops)
        return fail(TTN_EUNSUPPORTED, "fused plan exceeds its workspace bounds");
    for (const auto& ps : fp.passes)
        if (ps.mop_end - ps.mop_begin > ttn::FMAX_MOPS || ps.gate_end - ps.gate_begin > ttn::FMAX_GATES ||
            (ps.low && (ps.first_layout != 1 || ps.last_layout != 1)))
            return fail(TTN_EUNSUPPORTED, "fused pass program out of bounds");
    TTN_CUDA(cudaMemcpyAsync(P->ws + y.f_mops, fp.mops.data(), fp.mops.size() * sizeof(ttn::MicroOp), cudaMemcpyHostToDevice, st));
    TTN_CUDA(cudaMemcpyAsync(P->ws + y.f_gate_rc, fp.gate_rc.data(), fp.gate_rc.size() * 4, cudaMemcpyHostToDevice, st));
    ttn::FusedPrepParams q{};
    q.L = P->L; q.n_gates = (int)fp.gate_rc.size();
    q.gate_rc = reinterpret_cast<const int*>(P->ws + y.f_gate_rc);
    q.Jh = reinterpret_cast<const float*>(P->ws + y.Jh);
    q.Jv = reinterpret_cast<const float*>(P->ws + y.Jv);
    q.h = P->has_field ? reinterpret_cast<const float*>(P->ws + y.h) : nullptr;
    q.gate_k = reinterpret_cast<float*>(P->ws + y.f_gate_k);
    q.final_tab = reinterpret_cast<float*>(P->ws + y.f_final);
    const ttn::FusedPass& lastp = fp.passes.back();
    q.fin_low = lastp.low; q.fin_layout = lastp.last_layout; q.fin_a = lastp.a;
    if (P->i16 || P->z2) q.fin_a = lastp.low ? 0 : lastp.a - ((P->i16 && P->z2) ? 2 : 1);   // word digit / half-state digit
    q.col_off = P->z2 ? 1 : 0;
    long work = ttn::FFINAL_FLOATS; if (q.n_gates > work) work = q.n_gates;
    dim3 grid((unsigned)((work + 255) / 256), (unsigned)P->batch);
    if (P->i16) {
        ttn::fused16_prep_kernel<<<grid, 256, 0, st>>>(q);
        TTN_CUDA(cudaGetLastError());
        TTN_CUDA(cudaFuncSetAttribute(ttn::fused_pass_kernel<true, 1, false, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ttn::fsmem_bytes(true, 1)));
        TTN_CUDA(cudaFuncSetAttribute(ttn::fused_pass_kernel<true, 1, false, true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ttn::fsmem_bytes(true, 1)));
        TTN_CUDA(cudaFuncSetAttribute(ttn::fused_pass_kernel<true, 1, false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ttn::fsmem_bytes(true, 1)));
    TTN_CUDA(cudaFuncSetAttribute(ttn::fused_pass_kernel<true, 1, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ttn::fsmem_bytes(true, 1)));
        TTN_CUDA(cudaFuncSetAttribute(ttn::fused_pass_kernel<false, 1, false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ttn::fsmem_bytes(false, 1)));
    TTN_CUDA(cudaFuncSetAttribute(ttn::fused_pass_kernel<false, 1, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ttn::fsmem_bytes(false, 1)));
    } else {
        ttn::fused_prep_kernel<<<grid, 256, 0, st>>>(q);
    }
    TTN_CUDA(cudaGetLastError());
    TTN_CUDA(cudaFuncSetAttribute(ttn::fused_pass_kernel<true, 0, false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ttn::fsmem_bytes(true)));
    TTN_CUDA(cudaFuncSetAttribute(ttn::fused_pass_kernel<true, 0, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ttn::fsmem_bytes(true)));
    TTN_CUDA(cudaFuncSetAttribute(ttn::fused_pass_kernel<false, 0, false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ttn::fsmem_bytes(false)));
    TTN_CUDA(cudaFuncSetAttribute(ttn::fused_pass_kernel<false, 0, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ttn::fsmem_bytes(false)));
    TTN_CUDA(cudaFuncSetAttribute(ttn::fused_pass_kernel<true, 0, false, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ttn::fsmem_bytes(true)));
    TTN_CUDA(cudaFuncSetAttribute(ttn::fused_pass_kernel<true, 0, false, true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ttn::fsmem_bytes(true)));
    TTN_CUDA(cudaFuncSetAttribute(ttn::fused_sweep_kernel<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ttn::fsmem_bytes(true)));
    TTN_CUDA(cudaFuncSetAttribute(ttn::fused_pass_kernel<true, 0, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ttn::fsmem_bytes(true)));
    TTN_CUDA(cudaFuncSetAttribute(ttn::fused_pass_kernel<false, 0, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ttn::fsmem_bytes(false)));
    int dev = 0, sms = 0, per_sm = 0, per_sm2 = 0;
    TTN_CUDA(cudaGetDevice(&dev));
    TTN_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    TTN_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, ttn::fused_pass_kernel<true>, ttn::FWARPS_LOW * 32, ttn::fsmem_bytes(true)));
    TTN_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm2, ttn::fused_pass_kernel<false>, ttn::FWARPS_HIGH * 32, ttn::fsmem_bytes(false)));
    if (per_sm2 < per_sm) per_sm = per_sm2;
    if (per_sm < 1) return fail(TTN_ECUDA, "fused kernel does not fit on an SM");
    P->fused_grid = sms * per_sm;
    return TTN_OK;
}

// batches of small lattices walk all checkpoints of an instance in one CTA (backtrace_inst_kernel)
static bool backtrace_one_cta(int L, int batch, const DebugCfg& dbg, bool z2 = false) {
    return !z2 && L <= 18 && L <= ttn::BT_MAX_L && batch >= 32 && !dbg.bt_multi;
}

static ttn_status launch_backtrace(ttn_plan* P, cudaStream_t st) {
    {
        const Layout& y = P->lay;
        ttn::ArgmaxParams ap{};
        ap.L = P->L; ap.NS = y.NS; ap.nblk = y.amax_blocks;
        ap.c_stride = (unsigned long long)y.ck.n_buf * y.NS;
        ap.Jv = reinterpret_cast<const float*>(P->ws + y.Jv);
        ap.Jh = reinterpret_cast<const float*>(P->ws + y.Jh);
        ap.h = P->has_field ? reinterpret_cast<const float*>(P->ws + y.h) : nullptr;
        ap.s_next = ap.s_out = reinterpret_cast<unsigned long long*>(P->ws + y.out_s);
        ap.part_v = reinterpret_cast<float*>(P->ws + y.amax_v);
        ap.part_s = reinterpret_cast<unsigned long long*>(P->ws + y.amax_s);
        ap.v_out = reinterpret_cast<float*>(P->ws + y.out_x);
        ap.sigma = reinterpret_cast<signed char*>(P->ws + y.sigma);
        if (y.ck.k == 0 && backtrace_one_cta(P->L, P->batch, P->dbg, P->z2)) {
            // batches of small lattices: one CTA walks all L checkpoints of its instance
            ap.C = reinterpret_cast<const float*>(P->ws + y.ckpt);
            ttn::backtrace_inst_kernel<<<P->batch, ttn::BT_THREADS, 0, st>>>(ap);
            TTN_CUDA(cudaGetLastError());
            return TTN_OK;
        }
        auto bt_row = [&](int r, int slot) -> ttn_status {
            ap.r = r; ap.has_next = (r < P->L - 1);
            ap.C = reinterpret_cast<const float*>(P->ws + y.ckpt) + (unsigned long long)slot * y.NS;
            if (P->z2) ttn::argmax_partial_kernel<true><<<dim3(ap.nblk, P->batch), 256, 0, st>>>(ap);
            else ttn::argmax_partial_kernel<false><<<dim3(ap.nblk, P->batch), 256, 0, st>>>(ap);
            TTN_CUDA(cudaGetLastError());
            ttn::argmax_final_kernel<<<P->batch, 32, 0, st>>>(ap);
            TTN_CUDA(cudaGetLastError());
            return TTN_OK;
        };
        const CkptScheme& ck = y.ck;
        if (ck.k == 0) {
            for (int r = P->L - 1; r >= 0; --r) { ttn_status s = bt_row(r, r); if (s != TTN_OK) return s; }
            return TTN_OK;
        }
        // sqrt-spaced checkpoints: backtrack row b from its kept checkpoint, re-sweep rows a+1 .. b-1 from
        // C_a into the ring, backtrack through them and through row a, continue below a
        int b = P->L - 1;
        ttn_status s = bt_row(b, ck.stored_slot(b));
        if (s != TTN_OK) return s;
        while (b > 0) {
            const int a = ck.prev_stored(b);
            for (int r = a + 1; r < b; ++r) P->slot_of_row[r] = ck.ring_slot(a, r);
            for (int k = P->row_pass[a + 1]; k < P->row_pass[b]; ++k) {
                s = launch_fused_pass(P, P->fplan.passes[k], st, nullptr, 0, nullptr);
                if (s != TTN_OK) return s;
            }
            for (int r = b - 1; r >= a; --r) { s = bt_row(r, P->slot_of_row[r]); if (s != TTN_OK) return s; }
            for (int r = a + 1; r < b; ++r) P->slot_of_row[r] = -1;
            b = a;
        }
    }
    return TTN_OK;
}

extern "C" {

const char* ttn_last_error(void) { return g_err; }
int ttn_version(void) { return 100; }

size_t ttn_workspace_bytes(int q, int L, ttn_semiring mode, int batch, int want_config) {
    const bool count = (mode == TTN_COUNTING_F32_F64);
    if ((q != 2 && q != 3) || batch < 1 ||
        (mode != TTN_TROPICAL_F32 && mode != TTN_COUNTING_F32_F64 && mode != TTN_TROPICAL_I16)) return 0;
    if (mode == TTN_TROPICAL_I16 && (q != 2 || want_config)) return 0;
    if (!limits_ok(q, L, count, want_config != 0)) return 0;
    const DebugCfg dbg = read_debug();
    // (with h = 0 the calls may store the flip-reduced half-state: every field is then smaller; the Potts
    // calls always run on the colour-rotation-reduced third where it applies)
    return make_layout(q, L, count, want_config != 0, batch, dbg, mode == TTN_TROPICAL_I16 && i16_eligible(q, L, dbg),
                       z3_eligible(q, L, count, dbg)).total;
}

size_t ttn_workspace_bytes_h0(int q, int L, ttn_semiring mode, int batch, int want_config) {
    const size_t full = ttn_workspace_bytes(q, L, mode, batch, want_config);
    if (!full || q != 2) return full;
    const DebugCfg dbg = read_debug();
    const bool count = (mode == TTN_COUNTING_F32_F64);
    const ttn_call call = want_config ? TTN_CALL_CONFIG : (count ? TTN_CALL_COUNT : (mode == TTN_TROPICAL_I16 ? TTN_CALL_ENERGY_I16 : TTN_CALL_ENERGY));
    if (!z2_geom(q, L, call, false, dbg)) return full;
    return make_layout(q, L, count, want_config != 0, batch, dbg, mode == TTN_TROPICAL_I16 && i16_eligible(q, L, dbg), true).total;
}

long ttn_plan_describe(int q, int L, ttn_call call, char* buf, size_t n) {
    if ((q != 2 && q != 3) || !buf || n == 0) return -1;
    {   // the limits of the call kind, plain or *_Z2, as ttn_plan_create derives them; the flip reduction is Ising only
        const bool z2_kind = (call == TTN_CALL_ENERGY_Z2 || call == TTN_CALL_COUNT_Z2 || call == TTN_CALL_ENERGY_I16_Z2 ||
                              call == TTN_CALL_CONFIG_Z2);
        if (call < TTN_CALL_ENERGY || call > TTN_CALL_CONFIG_Z2) return -1;
        if (q == 3 && (z2_kind || call == TTN_CALL_ENERGY_I16)) return -1;
        const bool count = (call == TTN_CALL_COUNT || call == TTN_CALL_COUNT_Z2);
        const bool config = (call == TTN_CALL_CONFIG || call == TTN_CALL_CONFIG_Z2);
        if (!limits_ok(q, L, count, config)) return -1;
    }
    std::string s;
    const DebugCfg dbg = read_debug();
    if (call == TTN_CALL_ENERGY_Z2 || call == TTN_CALL_COUNT_Z2 || call == TTN_CALL_ENERGY_I16_Z2 || call == TTN_CALL_CONFIG_Z2) {
        // the schedules the calls run when h = 0
        if (const ttn::FusedGeom* G = z2_geom(q, L, call, false, dbg)) {
            ttn::FusedPlan fp;
            fp = call == TTN_CALL_CONFIG_Z2 ? ttn::make_fused_row_plan(L, ttn::FMAX_GATES, *G) : ttn::make_fused_plan(L, ttn::FMAX_GATES, *G);
            if (fp.ok) s = ttn::describe_fused(fp);
        }
        if (s.empty()) call = call == TTN_CALL_ENERGY_Z2 ? TTN_CALL_ENERGY : (call == TTN_CALL_COUNT_Z2 ? TTN_CALL_COUNT
                            : (call == TTN_CALL_CONFIG_Z2 ? TTN_CALL_CONFIG : TTN_CALL_ENERGY_I16));
    }
    if (call == TTN_CALL_ENERGY_I16 && i16_eligible(q, L, dbg)) {
        ttn::FusedPlan fp = ttn::make_fused_plan(L, ttn::FMAX_GATES, ttn::GEOM_I16);
        if (fp.ok) s = ttn::describe_fused(fp);
    }
    if (call == TTN_CALL_ENERGY_I16 && s.empty()) call = TTN_CALL_ENERGY;
    if (s.empty() && fused_eligible(q, L, call == TTN_CALL_COUNT, call == TTN_CALL_CONFIG, dbg)) {
        ttn::FusedPlan fp;
        // (ttn_ground_config on batches of small lattices: the merged plan of the one-launch sweep; a single
        // instance runs one pass per tile and row -- TTN_DEBUG_NOMERGE shows that schedule)
        if (call == TTN_CALL_CONFIG && ckpt_scheme(L, true, dbg).k == 0 && !dbg.nomerge && !dbg.nosweep && !dbg.nogroup)
            fp = ttn::make_fused_row_plan_merged(L, ttn::FMAX_GATES);
        if (!fp.ok)
            fp = call == TTN_CALL_COUNT ? ttn::make_fused_plan(L, ttn::FMAX_GATES, ttn::GEOM_COUNT)
               : call == TTN_CALL_CONFIG ? ttn::make_fused_row_plan(L, ttn::FMAX_GATES)
                                         : ttn::make_fused_plan(L, ttn::FMAX_GATES);
        if (fp.ok) s = ttn::describe_fused(fp);
    }
    if (s.empty()) s = ttn::describe(plan_for(q, L, call, /*has_field=*/q == 2, dbg));
    size_t m = s.size() < n - 1 ? s.size() : n - 1;
    memcpy(buf, s.data(), m);
    buf[m] = 0;
    return (long)s.size();
}

ttn_status ttn_plan_create(int q, int L, ttn_call call, const float* Jh, const float* Jv,
                           const float* h, int batch, void* workspace, size_t workspace_bytes,
                           void* stream, ttn_plan** out) {
    if (!out) return fail(TTN_EINVAL, "plan pointer is NULL");
    *out = nullptr;
    if (q != 2 && q != 3) return fail(TTN_EINVAL, "q must be 2 or 3");
    if (L < 1 || batch < 1) return fail(TTN_EINVAL, "L and batch must be >= 1");
    if (call != TTN_CALL_ENERGY && call != TTN_CALL_COUNT && call != TTN_CALL_CONFIG && call != TTN_CALL_ENERGY_I16 &&
        call != TTN_CALL_ENERGY_Z2 && call != TTN_CALL_COUNT_Z2 && call != TTN_CALL_ENERGY_I16_Z2 && call != TTN_CALL_CONFIG_Z2)
        return fail(TTN_EINVAL, "bad call kind");
    const bool want_z2 = (call == TTN_CALL_ENERGY_Z2 || call == TTN_CALL_COUNT_Z2 || call == TTN_CALL_ENERGY_I16_Z2 ||
                          call == TTN_CALL_CONFIG_Z2);
    const DebugCfg dbg = read_debug();
    bool i16 = false;
    const bool want_i16 = (call == TTN_CALL_ENERGY_I16 || call == TTN_CALL_ENERGY_I16_Z2);
    if (want_i16) {
        if (q != 2) return fail(TTN_EINVAL, "Tropical<i16> is an Ising call");
        i16 = i16_eligible(q, L, dbg);      // small lattices run the f32 path (identical results)
    }
    if (want_z2 && q != 2) return fail(TTN_EINVAL, "the flip reduction is an Ising call");
    if (L > 1 && (!Jh || !Jv)) return fail(TTN_EINVAL, "Jh/Jv is NULL");
    if (!workspace) return fail(TTN_EINVAL, "workspace is NULL");
    if (q == 3 && h) return fail(TTN_EINVAL, "the Potts variant takes no fields");
    const bool count = (call == TTN_CALL_COUNT || call == TTN_CALL_COUNT_Z2), config = (call == TTN_CALL_CONFIG || call == TTN_CALL_CONFIG_Z2);
    if (!limits_ok(q, L, count, config)) return fail(TTN_EUNSUPPORTED, "L=%d beyond the limits for this call", L);
    const size_t nh = (size_t)batch * L * (L - 1), nv = (size_t)batch * (L - 1) * L, nf = (size_t)batch * L * L;
    for (size_t i = 0; i < nh; ++i) if (!std::isfinite(Jh[i])) return fail(TTN_EINVAL, "non-finite Jh[%zu]", i);
    for (size_t i = 0; i < nv; ++i) if (!std::isfinite(Jv[i])) return fail(TTN_EINVAL, "non-finite Jv[%zu]", i);
    if (h) for (size_t i = 0; i < nf; ++i) if (!std::isfinite(h[i])) return fail(TTN_EINVAL, "non-finite h[%zu]", i);

    if (want_i16) {
        // exactness: integer-valued couplings whose absolute sum keeps every intermediate inside 16 bits
        for (int b = 0; b < batch; ++b) {
            double tot = 0.0;
            auto scan = [&](const float* a, size_t n_) -> bool {
                for (size_t i = 0; i < n_; ++i) { if (a[i] != std::nearbyint(a[i])) return false; tot += std::fabs((double)a[i]); }
                return true;
            };
            bool ok = scan(Jh + (size_t)b * L * (L - 1), (size_t)L * (L - 1)) && scan(Jv + (size_t)b * (L - 1) * L, (size_t)(L - 1) * L);
            if (ok && h) ok = scan(h + (size_t)b * L * L, (size_t)L * L);
            if (!ok) return fail(TTN_EINVAL, "Tropical<i16> needs integer-valued couplings (instance %d)", b);
            if (tot > 8000.0) return fail(TTN_EINVAL, "Tropical<i16>: sum of |couplings| = %.0f > 8000 (instance %d)", tot, b);
        }
    }
    // h = NULL or all zero: Eq. (1) PAPER.md:29 is invariant under the global flip -> half-state (planner.h)
    bool field = false;
    if (h) for (size_t i = 0; i < nf && !field; ++i) field = (h[i] != 0.0f);
    if (want_z2 && field) return fail(TTN_EINVAL, "the flip reduction needs h = 0");
    const ttn::FusedGeom* zg = z2_geom(q, L, call, field, dbg);
    const bool z3 = z3_eligible(q, L, count, dbg);
    if (want_z2) call = count ? TTN_CALL_COUNT : (config ? TTN_CALL_CONFIG : (want_i16 ? TTN_CALL_ENERGY_I16 : TTN_CALL_ENERGY));  // lattices too small for it run the plain sweep
    Layout lay = make_layout(q, L, count, config, batch, dbg, i16, zg != nullptr || z3);
    if (workspace_bytes < lay.total)
        return fail(TTN_ENOMEM, "workspace too small: %zu < %zu", workspace_bytes, lay.total);
    if ((uintptr_t)workspace % 256) return fail(TTN_EINVAL, "workspace must be 256-byte aligned");

    int dev = 0, major = 0;
    TTN_CUDA(cudaGetDevice(&dev));
    TTN_CUDA(cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev));
    if (major != 10) return fail(TTN_EUNSUPPORTED, "device compute capability %d.x is not sm_100", major);

    ttn_plan* P = new (std::nothrow) ttn_plan();
    if (!P) return fail(TTN_ENOMEM, "host allocation failed");
    P->q = q; P->L = L; P->batch = batch; P->call = call; P->count = count; P->config = config;
    P->has_field = (h != nullptr) && zg == nullptr;
    P->i16 = i16;
    P->z2 = zg != nullptr || z3;
    P->dbg = dbg;
    P->lay = lay;
    {
        cudaError_t ce = cudaDeviceGetAttribute(&P->sms, cudaDevAttrMultiProcessorCount, dev);
        if (ce != cudaSuccess) { delete P; return fail(TTN_ECUDA, "cudaDeviceGetAttribute failed: %s", cudaGetErrorString(ce)); }
    }
    P->ws = static_cast<unsigned char*>(workspace);
    // merged row passes (MC_CKPT) exist in the instance-group kernels only: batches of lattices whose passes all
    // run one CTA per instance group (the one-launch forward sweep)
    const bool merged_ok = lay.ck.k == 0 && !dbg.nomerge && !dbg.nosweep && !dbg.nogroup && batch >= 2 &&
                           ((lay.NS >> 12) < 12ull * 64ull);
    if (i16) {
        P->fplan = ttn::make_fused_plan(L, ttn::FMAX_GATES, zg ? *zg : ttn::GEOM_I16);
        P->fused = P->fplan.ok;
        if (!P->fused) { delete P; return fail(TTN_EUNSUPPORTED, "no Tropical<i16> schedule"); }
    } else if (zg) {
        if (config) P->fplan = ttn::make_fused_row_plan(L, ttn::FMAX_GATES, *zg);       // (no one-launch sweep for half-states)
        if (!config) P->fplan = ttn::make_fused_plan(L, ttn::FMAX_GATES, *zg);
        P->fused = P->fplan.ok;
        if (!P->fused) { delete P; return fail(TTN_EUNSUPPORTED, "no flip-reduced schedule"); }
    } else if (fused_eligible(q, L, count, config, dbg)) {
        if (config && merged_ok) { P->fplan = ttn::make_fused_row_plan_merged(L, ttn::FMAX_GATES); P->merged = P->fplan.ok; }
        if (!P->fplan.ok)
            P->fplan = count ? ttn::make_fused_plan(L, ttn::FMAX_GATES, ttn::GEOM_COUNT)
                     : config ? ttn::make_fused_row_plan(L, ttn::FMAX_GATES) : ttn::make_fused_plan(L, ttn::FMAX_GATES);
        P->fused = P->fplan.ok;
    }
    if (!P->fused) P->plan = plan_for(q, L, call, P->has_field, dbg);
    if (!P->fused && P->plan.passes.empty()) { delete P; return fail(TTN_EUNSUPPORTED, "planner produced no schedule"); }
    if (P->plan.ops.size() > (size_t)(L * L + 8)) { delete P; return fail(TTN_EUNSUPPORTED, "op list too long"); }
    if (!P->fused && z3 != P->plan.vcol) { delete P; return fail(TTN_EUNSUPPORTED, "planner / layout disagree on the Z3 reduction"); }

    // the +J constants factored out of the Ising gates (kernel comment at OP_GATE), in f64
    P->defer.assign(batch, 0.0);
    if (q == 2)
        for (int b = 0; b < batch; ++b) {
            double s = 0.0;
            for (int i = 0; i < (L - 1) * L; ++i) s += (double)Jv[(size_t)b * (L - 1) * L + i];
            P->defer[b] = s;
        }

    cudaStream_t st = static_cast<cudaStream_t>(stream);
    auto up = [&](size_t off, const void* src, size_t bytes) -> cudaError_t {
        if (!bytes) return cudaSuccess;
        return cudaMemcpyAsync(P->ws + off, src, bytes, cudaMemcpyHostToDevice, st);
    };
    cudaError_t e = up(lay.Jh, Jh, nh * 4);
    if (e == cudaSuccess) e = up(lay.Jv, Jv, nv * 4);
    if (e == cudaSuccess && h) e = up(lay.h, h, nf * 4);
    if (e == cudaSuccess) e = up(lay.ops, P->plan.ops.data(), P->plan.ops.size() * sizeof(ttn::Op));
    if (e != cudaSuccess) { delete P; return fail(TTN_ECUDA, "coupling upload failed: %s", cudaGetErrorString(e)); }

    for (int attempt = 0; P->fused && attempt < 2; ++attempt) {
        if (attempt == 1) {                 // the merged plan did not fit the one-launch sweep: one pass per tile and row
            P->fplan = ttn::make_fused_row_plan(L, ttn::FMAX_GATES);
            P->merged = false; P->sweep_grid = 0; P->sweep_params.clear();
            if (!P->fplan.ok) { delete P; return fail(TTN_EUNSUPPORTED, "no row-aligned schedule"); }
        }
        ttn_status fs = count ? setup_fcount(P, st) : setup_fused(P, st);
        if (fs != TTN_OK) { delete P; return fs; }
        const CkptScheme& ck = lay.ck;
        const bool bt1 = ck.k == 0 && backtrace_one_cta(L, batch, dbg, P->z2);
        P->launches = (int)P->fplan.passes.size() + (config ? (bt1 ? 1 : 2 * L) : 1);
        if (config) {
            // passes of row r (row 0 = the initialising pass), and where C_r lives during the forward sweep
            P->row_pass.assign(L + 1, 0);
            int row = 0;
            for (size_t i = 0; i < P->fplan.passes.size(); ++i)
                if (P->fplan.passes[i].dst_buf >= 0) { P->row_pass[++row] = (int)i + 1; }
            if (ck.k > 0 && row != L) { delete P; return fail(TTN_EUNSUPPORTED, "row-aligned plan is incomplete"); }
            P->slot_of_row.assign(L, -1);
            for (int r = 0; r < L; ++r) if (ck.stored(r)) P->slot_of_row[r] = ck.stored_slot(r);
            if (ck.k > 0)          // the backward pass re-sweeps every row that is not kept
                for (int r = 1; r < L; ++r) if (!ck.stored(r)) P->launches += P->row_pass[r + 1] - P->row_pass[r];
        }
        if (config && ck.k == 0 && !count && !P->i16 && !P->z2 && !dbg.nosweep && P->fplan.passes.size() <= (size_t)(4 * L + 8)) {
            // every pass in cta_per_inst mode: the pass table of fused_sweep_kernel (two instances per
            // CTA at a time where the constants of every pass fit, else one)
            std::vector<ttn::FusedParams> v(P->fplan.passes.size());
            unsigned grid = 0;
            bool ok = false;
            for (int K = 2; K >= 1 && !ok; --K) {
                ok = true;
                for (size_t i = 0; i < v.size() && ok; ++i)
                    ok = launch_fused_pass(P, P->fplan.passes[i], st, &v[i], K, &grid) == TTN_OK;
            }
            if (ok) {
                P->sweep_params = v; P->sweep_grid = (int)grid;
                cudaError_t ce = cudaMemcpyAsync(P->ws + lay.f_sweep, P->sweep_params.data(), v.size() * sizeof(ttn::FusedParams),
                                                 cudaMemcpyHostToDevice, st);
                if (ce != cudaSuccess) { delete P; return fail(TTN_ECUDA, "pass table upload failed: %s", cudaGetErrorString(ce)); }
                P->launches = 1 + (bt1 ? 1 : 2 * L);
            }
        }
        if (!(P->merged && P->sweep_grid == 0)) break;
    }
    if (!P->fused) {
        ttn::GenericPrepParams gp{};
        gp.q = q; gp.L = L; gp.n_ops = (int)P->plan.ops.size();
        gp.col_off = P->plan.vcol ? 1 : 0;
        gp.ops = reinterpret_cast<const ttn::Op*>(P->ws + lay.ops);
        gp.Jh = reinterpret_cast<const float*>(P->ws + lay.Jh);
        gp.Jv = reinterpret_cast<const float*>(P->ws + lay.Jv);
        gp.h = P->has_field ? reinterpret_cast<const float*>(P->ws + lay.h) : nullptr;
        gp.gate_k = reinterpret_cast<float*>(P->ws + lay.g_gate_k);
        gp.fin = reinterpret_cast<float*>(P->ws + lay.g_fin);
        long work = 2 * ttn::GMAX_L; if (gp.n_ops > work) work = gp.n_ops;
        ttn::generic_prep_kernel<<<dim3((unsigned)((work + 255) / 256), (unsigned)batch), 256, 0, st>>>(gp);
        cudaError_t pe = cudaGetLastError();
        if (pe != cudaSuccess) { delete P; return fail(TTN_ECUDA, "prep launch failed: %s", cudaGetErrorString(pe)); }
        P->launches = (int)P->plan.passes.size() + (config ? (lay.ck.k == 0 && backtrace_one_cta(L, batch, dbg) ? 1 : 2 * L) : 1);
    }
    *out = P;
    return TTN_OK;
}

ttn_status ttn_plan_launch(ttn_plan* P, void* stream) {
    if (!P) return fail(TTN_EINVAL, "plan is NULL");
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    if (P->fused) {
        const bool timing = P->dbg.timing != 0;                        // per-pass device times on stderr
        std::vector<cudaEvent_t> ev;
        if (timing) { ev.resize(P->fplan.passes.size() + 1); for (auto& e : ev) cudaEventCreate(&e); cudaEventRecord(ev[0], st); }
        // batches of small lattices, no reduction pass (ttn_ground_config): all passes in one launch
        if (P->sweep_grid > 0 && (!timing || P->merged)) {
            ttn::fused_sweep_kernel<0><<<(unsigned)P->sweep_grid, ttn::fwarps(true) * 32, ttn::fsmem_bytes(true), st>>>(
                reinterpret_cast<const ttn::FusedParams*>(P->ws + P->lay.f_sweep), (int)P->sweep_params.size());
            TTN_CUDA(cudaGetLastError());
            return launch_backtrace(P, st);
        }
        size_t k = 0;
        for (const ttn::FusedPass& ps : P->fplan.passes) {
            ttn_status s = P->count ? launch_fcount_pass(P, ps, st) : launch_fused_pass(P, ps, st);
            if (s != TTN_OK) return s;
            if (timing) cudaEventRecord(ev[++k], st);
        }
        if (timing) {
            cudaStreamSynchronize(st);
            for (size_t i = 0; i < P->fplan.passes.size(); ++i) {
                float ms = 0; cudaEventElapsedTime(&ms, ev[i], ev[i + 1]);
                const ttn::FusedPass& ps = P->fplan.passes[i];
                fprintf(stderr, "pass %2zu a=%2d low=%d gates=%3d rounds=%2d phases=%d : %.2f ms\n", i, ps.a, ps.low,
                        ps.gate_end - ps.gate_begin, ps.n_rounds, ps.n_phases, ms);
            }
            for (auto& e : ev) cudaEventDestroy(e);
        }
        if (P->config) return launch_backtrace(P, st);
        return TTN_OK;
    }
    const bool gtiming = P->dbg.timing != 0;                         // per-pass device times on stderr
    std::vector<cudaEvent_t> gev;
    if (gtiming) { gev.resize(P->plan.passes.size() + 1); for (auto& e : gev) cudaEventCreate(&e); cudaEventRecord(gev[0], st); }
    size_t gk = 0;
    for (const ttn::Pass& ps : P->plan.passes) {
        ttn_status s;
        if (P->q == 2) s = P->count ? launch_pass<2, true>(P, ps, st) : launch_pass<2, false>(P, ps, st);
        else s = P->count ? launch_pass<3, true>(P, ps, st) : launch_pass<3, false>(P, ps, st);
        if (s != TTN_OK) return s;
        if (gtiming) cudaEventRecord(gev[++gk], st);
    }
    if (gtiming) {
        cudaStreamSynchronize(st);
        for (size_t i = 0; i < P->plan.passes.size(); ++i) {
            float ms = 0; cudaEventElapsedTime(&ms, gev[i], gev[i + 1]);
            const ttn::Pass& ps = P->plan.passes[i];
            fprintf(stderr, "gpass %2zu lo=%d a=%d b=%d gates=%3d flags=%d : %.2f ms\n", i, ps.lo, ps.a, ps.b, ps.n_gates, ps.flags, ms);
        }
        for (auto& e : gev) cudaEventDestroy(e);
    }
    if (P->config) return launch_backtrace(P, st);
    return TTN_OK;
}

ttn_status ttn_plan_read(ttn_plan* P, void* stream, double* E0, double* degeneracy, int8_t* sigma) {
    if (!P) return fail(TTN_EINVAL, "plan is NULL");
    if (!E0) return fail(TTN_EINVAL, "E0 is NULL");
    if (P->count && !degeneracy) return fail(TTN_EINVAL, "degeneracy is NULL");
    if (!P->count && degeneracy) return fail(TTN_EINVAL, "degeneracy given for a non-counting plan");
    if (P->config && !sigma) return fail(TTN_EINVAL, "sigma is NULL");
    if (!P->config && sigma) return fail(TTN_EINVAL, "sigma given for a non-config plan");
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    std::vector<float> x(P->batch);
    TTN_CUDA(cudaMemcpyAsync(x.data(), P->ws + P->lay.out_x, (size_t)P->batch * 4, cudaMemcpyDeviceToHost, st));
    if (P->count)
        TTN_CUDA(cudaMemcpyAsync(degeneracy, P->ws + P->lay.out_n, (size_t)P->batch * 8, cudaMemcpyDeviceToHost, st));
    if (P->config)
        TTN_CUDA(cudaMemcpyAsync(sigma, P->ws + P->lay.sigma, (size_t)P->batch * P->L * P->L, cudaMemcpyDeviceToHost, st));
    TTN_CUDA(cudaStreamSynchronize(st));
    if (P->count && P->z2)                           // the stored half (third) holds one of every flip pair (rotation triple)
        for (int b = 0; b < P->batch; ++b) degeneracy[b] *= (P->q == 3 ? 3.0 : 2.0);
    for (int b = 0; b < P->batch; ++b) {
        double m = (double)x[b] + P->defer[b];      // max of -E
        E0[b] = (m == 0.0) ? 0.0 : -m;              // -0.0 -> +0.0
    }
    return TTN_OK;
}

void ttn_plan_destroy(ttn_plan* P) { delete P; }
int ttn_plan_num_launches(const ttn_plan* P) { return P ? P->launches : 0; }
int ttn_plan_num_passes(const ttn_plan* P) { return P ? (int)(P->fused ? P->fplan.passes.size() : P->plan.passes.size()) : 0; }
unsigned long long ttn_plan_state_elements(const ttn_plan* P) { return P ? P->lay.NS : 0ull; }

}  // extern "C"

static ttn_status one_call(int q, int L, ttn_call call, const float* Jh, const float* Jv, const float* h,
                           int batch, void* ws, size_t wsb, void* stream, double* E0, double* g, int8_t* sigma) {
    if (!E0) return fail(TTN_EINVAL, "E0 is NULL");
    if (call == TTN_CALL_COUNT && !g) return fail(TTN_EINVAL, "degeneracy is NULL");
    if (call == TTN_CALL_CONFIG && !sigma) return fail(TTN_EINVAL, "sigma is NULL");
    ttn_plan* P = nullptr;
    ttn_status s = ttn_plan_create(q, L, call, Jh, Jv, h, batch, ws, wsb, stream, &P);
    if (s != TTN_OK) return s;
    s = ttn_plan_launch(P, stream);
    if (s == TTN_OK) s = ttn_plan_read(P, stream, E0, g, sigma);
    else cudaStreamSynchronize(static_cast<cudaStream_t>(stream));
    ttn_plan_destroy(P);
    return s;
}

extern "C" {

ttn_status ttn_sweep_energy(int L, const float* Jh, const float* Jv, const float* h, int batch,
                            void* ws, size_t wsb, void* stream, double* E0) {
    return one_call(2, L, TTN_CALL_ENERGY, Jh, Jv, h, batch, ws, wsb, stream, E0, nullptr, nullptr);
}
ttn_status ttn_sweep_energy_i16(int L, const float* Jh, const float* Jv, const float* h, int batch,
                                void* ws, size_t wsb, void* stream, double* E0) {
    return one_call(2, L, TTN_CALL_ENERGY_I16, Jh, Jv, h, batch, ws, wsb, stream, E0, nullptr, nullptr);
}
ttn_status ttn_sweep_count(int L, const float* Jh, const float* Jv, const float* h, int batch,
                           void* ws, size_t wsb, void* stream, double* E0, double* g) {
    return one_call(2, L, TTN_CALL_COUNT, Jh, Jv, h, batch, ws, wsb, stream, E0, g, nullptr);
}
ttn_status ttn_ground_config(int L, const float* Jh, const float* Jv, const float* h, int batch,
                             void* ws, size_t wsb, void* stream, double* E0, int8_t* sigma) {
    return one_call(2, L, TTN_CALL_CONFIG, Jh, Jv, h, batch, ws, wsb, stream, E0, nullptr, sigma);
}
ttn_status ttn_potts3_sweep_energy(int L, const float* Jh, const float* Jv, int batch, void* ws,
                                   size_t wsb, void* stream, double* E0) {
    return one_call(3, L, TTN_CALL_ENERGY, Jh, Jv, nullptr, batch, ws, wsb, stream, E0, nullptr, nullptr);
}
ttn_status ttn_potts3_sweep_count(int L, const float* Jh, const float* Jv, int batch, void* ws,
                                  size_t wsb, void* stream, double* E0, double* g) {
    return one_call(3, L, TTN_CALL_COUNT, Jh, Jv, nullptr, batch, ws, wsb, stream, E0, g, nullptr);
}

// ---- chimera graph, Tropical<i16> (ttn_chimera.cuh) ---------------------------
}  // extern "C"

// ---- chimera, M >= 4: the 16^M state of ttn_chimera2.cuh.  The horizontal couplings of a column are one
// gate row of a 4M-column Ising lattice in Tropical<i16>: an internal plan drives the fused pass kernels.
namespace {
constexpr int CH2_MIN_M = 4;
struct Chimera2Layout {
    Layout lay;                 // of the internal Ising plan (state, programs; batch 1)
    size_t fJh = 0, fJv = 0, gate_k = 0, final_tab = 0, tables = 0, out = 0, total = 0;
};
Chimera2Layout chimera2_layout(int M, int N, const DebugCfg& dbg) {
    Chimera2Layout c;
    const int NB = 4 * M, cols = N > 1 ? N - 1 : 1;
    DebugCfg d = dbg; d.fused = 1;           // the gate rows always run on the fused pass kernels, whatever TTN_DEBUG_FUSED says
    c.lay = make_layout(2, NB, false, false, 1, d, /*i16=*/true, false);
    size_t off = c.lay.total;
    auto take = [&](size_t bytes) { size_t o = off; off = align_up(off + bytes); return o; };
    c.fJh = take((size_t)cols * NB * (NB - 1) * 4 + 4);           // fake couplings, one "instance" per column
    c.fJv = take((size_t)cols * (NB - 1) * NB * 4 + 4);
    c.gate_k = take((size_t)cols * NB * 8 * 4);
    c.final_tab = take((size_t)cols * ttn::FFINAL_FLOATS * 4);
    c.tables = take((size_t)M * N * 128 * 4);
    c.out = take(256);
    c.total = off;
    return c;
}
}  // namespace

static ttn_status chimera2_sweep(int M, int N, const float* K, const float* Jv, const float* Jh, void* ws,
                                 size_t wsb, void* stream, double* E0, const DebugCfg& dbg);

// counting: rows of cells are padded with coupling-free cells up to CHC_MIN_M (each adds 8 free spins: x 2^8)
namespace {
constexpr int CHC_MIN_M = 3;
struct ChimeraCountLayout {
    Layout lay;                 // of the internal counting Ising plan (x, n, programs; batch 1)
    size_t fJh = 0, fJv = 0, gate_k = 0, final_tab = 0, tables = 0, total = 0;
};
ChimeraCountLayout chimera_count_layout(int Mp, int N, const DebugCfg& dbg) {
    ChimeraCountLayout c;
    const int NB = 4 * Mp, cols = N > 1 ? N - 1 : 1;
    DebugCfg d = dbg; d.fused = 1;           // (as chimera2_layout)
    c.lay = make_layout(2, NB, true, false, 1, d, false, false);
    size_t off = c.lay.total;
    auto take = [&](size_t bytes) { size_t o = off; off = align_up(off + bytes); return o; };
    c.fJh = take((size_t)cols * NB * (NB - 1) * 4 + 4);
    c.fJv = take((size_t)cols * (NB - 1) * NB * 4 + 4);
    c.gate_k = take((size_t)cols * NB * 8 * 4);
    c.final_tab = take((size_t)cols * ttn::CFINAL_FLOATS * 4);
    c.tables = take((size_t)Mp * N * 256 * 4);
    c.total = off;
    return c;
}
}  // namespace

extern "C" {

size_t ttn_chimera_count_workspace_bytes(int M, int N) {
    if (M < 1 || M > 8 || N < 1 || N > 64) return 0;
    return chimera_count_layout(M < CHC_MIN_M ? CHC_MIN_M : M, N, read_debug()).total;
}

size_t ttn_chimera_workspace_bytes(int M, int N) {
    if (M < 1 || M > 8 || N < 1 || N > 64) return 0;
    if (M >= CH2_MIN_M) return chimera2_layout(M, N, read_debug()).total;
    return align_up((size_t)2 << (4 * M + 4)) + align_up((size_t)M * N * 128 * 4) + 256;
}

ttn_status ttn_chimera_sweep_energy_i16(int M, int N, const float* K, const float* Jv, const float* Jh,
                                        void* ws, size_t wsb, void* stream, double* E0) {
    if (M < 1 || N < 1 || !K || !E0 || !ws || (M > 1 && !Jv) || (N > 1 && !Jh)) return fail(TTN_EINVAL, "bad argument");
    if (M > 8 || N > 64) return fail(TTN_EUNSUPPORTED, "chimera: M <= 8 rows of cells (state 2^(4M+4) int16), N <= 64");
    const size_t need = ttn_chimera_workspace_bytes(M, N);
    if (wsb < need) return fail(TTN_ENOMEM, "workspace too small: %zu < %zu", wsb, need);
    if ((uintptr_t)ws % 256) return fail(TTN_EINVAL, "workspace must be 256-byte aligned");
    const DebugCfg dbg = read_debug();
    // integer-valued couplings whose absolute sum fits 16 bits with room (as ttn_sweep_energy_i16)
    double total = 0;
    auto scan = [&](const float* a, size_t n) {
        for (size_t i = 0; i < n; ++i) {
            const double x = (double)a[i];
            if (!std::isfinite(x) || x != std::nearbyint(x)) return false;
            total += std::fabs(x);
        }
        return true;
    };
    if (!scan(K, (size_t)M * N * 16) || (M > 1 && !scan(Jv, (size_t)(M - 1) * N * 4)) || (N > 1 && !scan(Jh, (size_t)M * (N - 1) * 4)))
        return fail(TTN_EINVAL, "chimera i16: couplings must be finite integers");
    if (total > 8000.0) return fail(TTN_EINVAL, "chimera i16: sum |J| = %.0f exceeds 8000", total);
    if (M >= CH2_MIN_M) return chimera2_sweep(M, N, K, Jv, Jh, ws, wsb, stream, E0, dbg);
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    unsigned char* base = static_cast<unsigned char*>(ws);
    unsigned* state = reinterpret_cast<unsigned*>(base);
    const size_t state_bytes = (size_t)2 << (4 * M + 4);
    unsigned* tables = reinterpret_cast<unsigned*>(base + align_up(state_bytes));
    int* d_out = reinterpret_cast<int*>(base + align_up(state_bytes) + align_up((size_t)M * N * 128 * 4));
    // the cells' tables B(u, v) = sum_kl K[k][l] s_k(v) s_l(u), packed over the lowest bit of v
    std::vector<unsigned> tab((size_t)M * N * 128);
    for (int r = 0; r < M; ++r)
        for (int c = 0; c < N; ++c) {
            const float* Kc = K + ((size_t)r * N + c) * 16;
            for (int u = 0; u < 16; ++u)
                for (int j = 0; j < 8; ++j) {
                    int val[2];
                    for (int hlf = 0; hlf < 2; ++hlf) {
                        const int v = 2 * j + hlf;
                        int acc = 0;
                        for (int k = 0; k < 4; ++k)
                            for (int l = 0; l < 4; ++l)
                                acc += (int)Kc[k * 4 + l] * (((v >> k) & 1) ? -1 : 1) * (((u >> l) & 1) ? -1 : 1);
                        val[hlf] = acc;
                    }
                    tab[(((size_t)r * N + c) * 16 + u) * 8 + j] = ((unsigned)val[0] & 0xffffu) | ((unsigned)val[1] << 16);
                }
        }
    TTN_CUDA(cudaMemcpyAsync(tables, tab.data(), tab.size() * 4, cudaMemcpyHostToDevice, st));
    const int int_min = -2147483647 - 1;
    TTN_CUDA(cudaMemcpyAsync(d_out, &int_min, sizeof(int), cudaMemcpyHostToDevice, st));
    // a gate is applied as max(A, B - 2J); its common + J is summed here and added to the maximum
    long shift = 0;
    auto pack = [&](float J) { shift += (long)J; const unsigned h = (unsigned)(-2 * (int)J) & 0xffffu; return h | (h << 16); };
    ttn::ChimeraCellParams q;
    q.state = state;
    q.groups = 1ull << (4 * M - 4);
    unsigned long long blocks = (q.groups + ttn::CH_THREADS - 1) / ttn::CH_THREADS;
    {   // a CTA walks its groups with the stride of the grid; 512 CTAs per SM measured best at 8 x 8
        // cells (per SM 8 / 32 / 64 / 128 / 512 CTAs: 3.27 / 3.24 / 3.19 / 3.15 / 3.12 s; one group per
        // thread, i.e. 2^23 CTAs: 3.61 s)
        int dev = 0, sms = 0, major = 0;
        const int per_sm = dbg.ch_persm;
        TTN_CUDA(cudaGetDevice(&dev));
        TTN_CUDA(cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev));
        if (major != 10) return fail(TTN_EUNSUPPORTED, "device compute capability %d.x is not sm_100", major);
        TTN_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
        const unsigned long long cap = (unsigned long long)sms * (unsigned long long)per_sm;
        if (blocks > cap) blocks = cap;
    }
    for (int c = 0; c < N; ++c)
        for (int r = 0; r < M; ++r) {
            q.p = 4 + 4 * r;
            q.init = (c == 0 && r == 0) ? 1 : 0;      // write-only first pass: every element is written
            for (int l = 0; l < 4; ++l) q.ju[l] = c > 0 ? pack(Jh[((size_t)r * (N - 1) + (c - 1)) * 4 + l]) : 0u;
            for (int k = 0; k < 4; ++k) q.jv[k] = r > 0 ? pack(Jv[((size_t)(r - 1) * N + c) * 4 + k]) : 0u;
            q.table = tables + ((size_t)r * N + c) * 128;
            if (r == 0 && q.groups >= 32 && !dbg.ch_nocell0) {
                const unsigned long long tiles = q.groups >> 5, wpb = ttn::CH_THREADS / 32;
                const unsigned long long b0 = (tiles + wpb - 1) / wpb;
                ttn::chimera_cell0_kernel<<<(unsigned)(b0 < blocks ? b0 : blocks), ttn::CH_THREADS, 0, st>>>(q);
            } else {
                ttn::chimera_cell_kernel<<<(unsigned)blocks, ttn::CH_THREADS, 0, st>>>(q);
            }
            TTN_CUDA(cudaGetLastError());
        }
    const unsigned long long quads = 1ull << (4 * M + 1);           // uint4 = 8 elements
    const unsigned rb = (unsigned)(quads / 256 < 148ull * 8 ? (quads + 255) / 256 : 148ull * 8);
    ttn::chimera_max_kernel<<<rb, 256, 0, st>>>(reinterpret_cast<const uint4*>(state), quads, d_out);
    TTN_CUDA(cudaGetLastError());
    int mx = 0;
    TTN_CUDA(cudaMemcpyAsync(&mx, d_out, sizeof(int), cudaMemcpyDeviceToHost, st));
    TTN_CUDA(cudaStreamSynchronize(st));
    const long top = (long)mx + shift;
    *E0 = top == 0 ? 0.0 : -(double)top;
    return TTN_OK;
}

}  // extern "C"

// The cells' tables B(u, v) = sum_kl K[k][l] s_k(v) s_l(u), packed over the lowest bit of v: [cell][16 u][8 words]
static void chimera_tables(int M, int N, const float* K, bool column_major, std::vector<unsigned>& tab) {
    tab.assign((size_t)M * N * 128, 0u);
    for (int r = 0; r < M; ++r)
        for (int c = 0; c < N; ++c) {
            const float* Kc = K + ((size_t)r * N + c) * 16;
            const size_t cell = column_major ? (size_t)c * M + r : (size_t)r * N + c;
            for (int u = 0; u < 16; ++u)
                for (int j = 0; j < 8; ++j) {
                    int val[2];
                    for (int hlf = 0; hlf < 2; ++hlf) {
                        const int v = 2 * j + hlf;
                        int acc = 0;
                        for (int k = 0; k < 4; ++k)
                            for (int l = 0; l < 4; ++l)
                                acc += (int)Kc[k * 4 + l] * (((v >> k) & 1) ? -1 : 1) * (((u >> l) & 1) ? -1 : 1);
                        val[hlf] = acc;
                    }
                    tab[(cell * 16 + u) * 8 + j] = ((unsigned)val[0] & 0xffffu) | ((unsigned)val[1] << 16);
                }
        }
}

static ttn_status chimera2_sweep(int M, int N, const float* K, const float* Jv, const float* Jh, void* ws,
                                 size_t wsb, void* stream, double* E0, const DebugCfg& dbg) {
    (void)wsb;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const int NB = 4 * M, cols = N - 1;
    const Chimera2Layout cl = chimera2_layout(M, N, dbg);
    unsigned char* base = static_cast<unsigned char*>(ws);
    int dev = 0, major = 0, sms = 0;
    TTN_CUDA(cudaGetDevice(&dev));
    TTN_CUDA(cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev));
    if (major != 10) return fail(TTN_EUNSUPPORTED, "device compute capability %d.x is not sm_100", major);
    TTN_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    // ---- tables of the cells, column-major, and the deferred constant of every gate
    std::vector<unsigned> tab;
    chimera_tables(M, N, K, /*column_major=*/true, tab);
    TTN_CUDA(cudaMemcpyAsync(base + cl.tables, tab.data(), tab.size() * 4, cudaMemcpyHostToDevice, st));
    const int int_min = -2147483647 - 1;
    TTN_CUDA(cudaMemcpyAsync(base + cl.out, &int_min, sizeof(int), cudaMemcpyHostToDevice, st));
    long shift = 0;
    for (size_t i = 0; i < (size_t)(M - 1) * N * 4; ++i) shift += (long)Jv[i];
    for (size_t i = 0; i < (size_t)M * (N - 1) * 4; ++i) shift += (long)Jh[i];
    // ---- the internal Ising plan: one gate row over the 4M bits of u, Tropical<i16>
    ttn_plan P{};
    P.q = 2; P.L = NB; P.batch = 1; P.call = TTN_CALL_ENERGY_I16; P.count = false; P.config = false; P.has_field = false;
    P.fused = true; P.i16 = true; P.z2 = false; P.dbg = dbg; P.lay = cl.lay; P.ws = base; P.sms = sms;
    std::vector<float> fJv, fJh;
    if (cols > 0) {
        P.fplan = ttn::make_gate_row_plan(NB, NB - 1, ttn::FMAX_GATES, ttn::GEOM_I16);     // the top bit: column kernel
        if (!P.fplan.ok) return fail(TTN_EUNSUPPORTED, "chimera: no gate-row schedule for %d bits", NB);
        // fake lattice per column c >= 1: Jv[0][4 r + l] = Jh_chimera[r][c-1][l], everything else 0, so that the
        // conjugation A_0 of the diagonal frame is the identity and gate (1, b) is the plain gate (A2) on bit b
        fJv.assign((size_t)cols * (NB - 1) * NB, 0.f);
        fJh.assign((size_t)cols * NB * (NB - 1), 0.f);
        for (int c = 1; c < N; ++c)
            for (int r = 0; r < M; ++r)
                for (int l = 0; l < 4; ++l)
                    fJv[(size_t)(c - 1) * (NB - 1) * NB + 4 * r + l] = Jh[((size_t)r * (N - 1) + (c - 1)) * 4 + l];
        TTN_CUDA(cudaMemcpyAsync(base + cl.fJv, fJv.data(), fJv.size() * 4, cudaMemcpyHostToDevice, st));
        TTN_CUDA(cudaMemcpyAsync(base + cl.fJh, fJh.data(), fJh.size() * 4, cudaMemcpyHostToDevice, st));
        const ttn::FusedPlan& fp = P.fplan;
        if ((int)fp.gate_rc.size() > cl.lay.f_max_gates || (int)fp.mops.size() > cl.lay.f_max_mops)
            return fail(TTN_EUNSUPPORTED, "chimera: gate-row plan exceeds its workspace bounds");
        TTN_CUDA(cudaMemcpyAsync(base + cl.lay.f_mops, fp.mops.data(), fp.mops.size() * sizeof(ttn::MicroOp), cudaMemcpyHostToDevice, st));
        TTN_CUDA(cudaMemcpyAsync(base + cl.lay.f_gate_rc, fp.gate_rc.data(), fp.gate_rc.size() * 4, cudaMemcpyHostToDevice, st));
        ttn::FusedPrepParams q{};
        q.L = NB; q.n_gates = (int)fp.gate_rc.size();
        q.gate_rc = reinterpret_cast<const int*>(base + cl.lay.f_gate_rc);
        q.Jh = reinterpret_cast<const float*>(base + cl.fJh);
        q.Jv = reinterpret_cast<const float*>(base + cl.fJv);
        q.h = nullptr;
        q.gate_k = reinterpret_cast<float*>(base + cl.gate_k);
        q.final_tab = reinterpret_cast<float*>(base + cl.final_tab);
        q.fin_low = 1; q.fin_layout = 1; q.fin_a = 0; q.col_off = 0;
        long work = ttn::FFINAL_FLOATS; if (q.n_gates > work) work = q.n_gates;
        ttn::fused16_prep_kernel<<<dim3((unsigned)((work + 255) / 256), (unsigned)cols), 256, 0, st>>>(q);
        TTN_CUDA(cudaGetLastError());
        TTN_CUDA(cudaFuncSetAttribute(ttn::fused_pass_kernel<true, 1, false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ttn::fsmem_bytes(true, 1)));
        TTN_CUDA(cudaFuncSetAttribute(ttn::fused_pass_kernel<false, 1, false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ttn::fsmem_bytes(false, 1)));
        P.fused_grid = sms;
    }
    ttn::ChimeraColumnParams cp{};
    cp.state = reinterpret_cast<unsigned*>(base + cl.lay.x);
    cp.M = M;
    cp.tiles = 1ull << (NB - 12);
    cp.out = reinterpret_cast<int*>(base + cl.out);
    const unsigned long long need = ((cp.tiles >> 1) + ttn::CH2_WARPS - 1) / ttn::CH2_WARPS;      // a warp takes a tile pair
    const unsigned cgrid = (unsigned)(need < 2ull * sms ? need : 2ull * sms);
    std::vector<cudaEvent_t> ev;               // TTN_DEBUG_TIMING: per-launch device times on stderr
    auto stamp = [&]() { if (dbg.timing) { cudaEvent_t e; cudaEventCreate(&e); cudaEventRecord(e, st); ev.push_back(e); } };
    stamp();
    for (int c = 0; c < N; ++c) {
        if (c > 0) {
            // the column's constants: instance c - 1 of the prep kernel's output
            P.lay.f_gate_k = cl.gate_k + (size_t)(c - 1) * P.fplan.gate_rc.size() * 32;
            for (const ttn::FusedPass& ps : P.fplan.passes) {
                ttn_status s = launch_fused_pass(&P, ps, st);
                if (s != TTN_OK) return s;
                stamp();
            }
        }
        cp.init = (c == 0); cp.reduce = (c == N - 1);
        {
            const int J = c > 0 ? (int)Jh[((size_t)(M - 1) * (N - 1) + (c - 1)) * 4 + 3] : 0;
            const unsigned h = (unsigned)(-2 * J) & 0xffffu;
            cp.ju_top = h | (h << 16);
        }
        cp.tables = reinterpret_cast<const unsigned*>(base + cl.tables) + (size_t)c * M * 128;
        for (int r = 0; r < 8; ++r)
            for (int k = 0; k < 4; ++k) {
                const int J = (r >= 1 && r < M) ? (int)Jv[((size_t)(r - 1) * N + c) * 4 + k] : 0;
                const unsigned h = (unsigned)(-2 * J) & 0xffffu;
                cp.jv[r][k] = h | (h << 16);
            }
        ttn::chimera_column_kernel<<<cgrid, ttn::CH2_WARPS * 32, 0, st>>>(cp);
        TTN_CUDA(cudaGetLastError());
        stamp();
    }
    if (dbg.timing) {
        cudaStreamSynchronize(st);
        for (size_t i = 1; i < ev.size(); ++i) { float ms = 0; cudaEventElapsedTime(&ms, ev[i - 1], ev[i]); fprintf(stderr, "chimera launch %2zu : %.2f ms\n", i - 1, ms); }
        for (auto& e : ev) cudaEventDestroy(e);
    }
    int mx = 0;
    TTN_CUDA(cudaMemcpyAsync(&mx, base + cl.out, sizeof(int), cudaMemcpyDeviceToHost, st));
    TTN_CUDA(cudaStreamSynchronize(st));
    const long top = (long)mx + shift;
    *E0 = top == 0 ? 0.0 : -(double)top;
    return TTN_OK;
}

// ---- chimera, CountingTropical (ttn_chimera2.cuh, second half) ----------------------------------------
extern "C" ttn_status ttn_chimera_sweep_count(int M, int N, const float* K, const float* Jv, const float* Jh,
                                               void* ws, size_t wsb, void* stream, double* E0, double* degeneracy) {
    if (M < 1 || N < 1 || !K || !E0 || !degeneracy || !ws || (M > 1 && !Jv) || (N > 1 && !Jh)) return fail(TTN_EINVAL, "bad argument");
    if (M > 8 || N > 64) return fail(TTN_EUNSUPPORTED, "chimera: M <= 8 rows of cells, N <= 64");
    const size_t need = ttn_chimera_count_workspace_bytes(M, N);
    if (wsb < need) return fail(TTN_ENOMEM, "workspace too small: %zu < %zu", wsb, need);
    if ((uintptr_t)ws % 256) return fail(TTN_EINVAL, "workspace must be 256-byte aligned");
    const DebugCfg dbg = read_debug();
    double total = 0;
    auto scan = [&](const float* a, size_t n) {
        for (size_t i = 0; i < n; ++i) {
            const double x = (double)a[i];
            if (!std::isfinite(x) || x != std::nearbyint(x)) return false;
            total += std::fabs(x);
        }
        return true;
    };
    if (!scan(K, (size_t)M * N * 16) || (M > 1 && !scan(Jv, (size_t)(M - 1) * N * 4)) || (N > 1 && !scan(Jh, (size_t)M * (N - 1) * 4)))
        return fail(TTN_EINVAL, "chimera count: couplings must be finite integers");
    if (total > 4.0e6) return fail(TTN_EINVAL, "chimera count: sum |J| = %.0f exceeds the exact f32 integer range", total);
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const int Mp = M < CHC_MIN_M ? CHC_MIN_M : M, NB = 4 * Mp, cols = N - 1;
    const ChimeraCountLayout cl = chimera_count_layout(Mp, N, dbg);
    unsigned char* base = static_cast<unsigned char*>(ws);
    int dev = 0, major = 0, sms = 0;
    TTN_CUDA(cudaGetDevice(&dev));
    TTN_CUDA(cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev));
    if (major != 10) return fail(TTN_EUNSUPPORTED, "device compute capability %d.x is not sm_100", major);
    TTN_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    // ---- tables B_r(u, v) of every cell as floats, column-major [c][r][16 u][16 v]; padded rows are zero
    std::vector<float> tab((size_t)Mp * N * 256, 0.f);
    for (int r = 0; r < M; ++r)
        for (int c = 0; c < N; ++c) {
            const float* Kc = K + ((size_t)r * N + c) * 16;
            float* out = tab.data() + ((size_t)c * Mp + r) * 256;
            for (int u = 0; u < 16; ++u)
                for (int v = 0; v < 16; ++v) {
                    int acc = 0;
                    for (int k = 0; k < 4; ++k)
                        for (int l = 0; l < 4; ++l)
                            acc += (int)Kc[k * 4 + l] * (((v >> k) & 1) ? -1 : 1) * (((u >> l) & 1) ? -1 : 1);
                    out[u * 16 + v] = (float)acc;
                }
        }
    TTN_CUDA(cudaMemcpyAsync(base + cl.tables, tab.data(), tab.size() * 4, cudaMemcpyHostToDevice, st));
    double shift = 0;
    for (size_t i = 0; i < (size_t)(M - 1) * N * 4; ++i) shift += (double)Jv[i];
    for (size_t i = 0; i < (size_t)M * (N - 1) * 4; ++i) shift += (double)Jh[i];
    // ---- the internal counting Ising plan: one gate row over the 4 Mp bits of u
    ttn_plan P{};
    P.q = 2; P.L = NB; P.batch = 1; P.call = TTN_CALL_COUNT; P.count = true; P.config = false; P.has_field = false;
    P.fused = true; P.i16 = false; P.z2 = false; P.dbg = dbg; P.lay = cl.lay; P.ws = base; P.sms = sms;
    std::vector<float> fJv, fJh;
    if (cols > 0) {
        P.fplan = ttn::make_gate_row_plan(NB, NB, ttn::FMAX_GATES, ttn::GEOM_COUNT);
        if (!P.fplan.ok) return fail(TTN_EUNSUPPORTED, "chimera count: no gate-row schedule for %d bits", NB);
        fJv.assign((size_t)cols * (NB - 1) * NB, 0.f);
        fJh.assign((size_t)cols * NB * (NB - 1), 0.f);
        for (int c = 1; c < N; ++c)
            for (int r = 0; r < M; ++r)
                for (int l = 0; l < 4; ++l)
                    fJv[(size_t)(c - 1) * (NB - 1) * NB + 4 * r + l] = Jh[((size_t)r * (N - 1) + (c - 1)) * 4 + l];
        TTN_CUDA(cudaMemcpyAsync(base + cl.fJv, fJv.data(), fJv.size() * 4, cudaMemcpyHostToDevice, st));
        TTN_CUDA(cudaMemcpyAsync(base + cl.fJh, fJh.data(), fJh.size() * 4, cudaMemcpyHostToDevice, st));
        const ttn::FusedPlan& fp = P.fplan;
        if ((int)fp.gate_rc.size() > cl.lay.f_max_gates || (int)fp.mops.size() > cl.lay.f_max_mops)
            return fail(TTN_EUNSUPPORTED, "chimera count: gate-row plan exceeds its workspace bounds");
        TTN_CUDA(cudaMemcpyAsync(base + cl.lay.f_mops, fp.mops.data(), fp.mops.size() * sizeof(ttn::MicroOp), cudaMemcpyHostToDevice, st));
        TTN_CUDA(cudaMemcpyAsync(base + cl.lay.f_gate_rc, fp.gate_rc.data(), fp.gate_rc.size() * 4, cudaMemcpyHostToDevice, st));
        ttn::CountPrepParams q{};
        q.L = NB; q.n_gates = (int)fp.gate_rc.size();
        q.gate_rc = reinterpret_cast<const int*>(base + cl.lay.f_gate_rc);
        q.Jh = reinterpret_cast<const float*>(base + cl.fJh);
        q.Jv = reinterpret_cast<const float*>(base + cl.fJv);
        q.h = nullptr;
        q.gate_k = reinterpret_cast<float*>(base + cl.gate_k);
        q.final_tab = reinterpret_cast<float*>(base + cl.final_tab);
        q.fin_low = 1; q.fin_layout = 1; q.fin_a = 0; q.col_off = 0;
        long work = ttn::CFINAL_FLOATS; if (q.n_gates > work) work = q.n_gates;
        ttn::fcount_prep_kernel<<<dim3((unsigned)((work + 255) / 256), (unsigned)cols), 256, 0, st>>>(q);
        TTN_CUDA(cudaGetLastError());
        TTN_CUDA(cudaFuncSetAttribute(ttn::fcount_pass_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ttn::csmem_bytes()));
        TTN_CUDA(cudaFuncSetAttribute(ttn::fcount_pass_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ttn::csmem_bytes()));
        P.fused_grid = sms;
    }
    ttn::ChimeraCountParams cp{};
    cp.x = reinterpret_cast<float*>(base + cl.lay.x);
    cp.n = reinterpret_cast<double*>(base + cl.lay.n);
    cp.M = Mp;
    cp.tiles = 1ull << (NB - 12);
    cp.part_x = reinterpret_cast<float*>(base + cl.lay.part_x);
    cp.part_n = reinterpret_cast<double*>(base + cl.lay.part_n);
    // every padded cell carries 8 free spins, a factor 2^8 on the count per column: taken out column by column (an
    // exact power-of-two scaling) so that the running count never holds 2^(8 N (Mp - M)) -- 2^1024 at M = 1, N = 64
    cp.n_scale = std::ldexp(1.0, -8 * (Mp - M));
    const unsigned long long needc = (cp.tiles + ttn::CH2C_WARPS - 1) / ttn::CH2C_WARPS;
    const unsigned cgrid = (unsigned)(needc < (unsigned long long)sms ? needc : (unsigned long long)sms);
    if ((unsigned long long)cgrid > cl.lay.max_tiles) return fail(TTN_EUNSUPPORTED, "chimera count: partials do not fit");
    for (int c = 0; c < N; ++c) {
        if (c > 0) {
            P.lay.f_gate_k = cl.gate_k + (size_t)(c - 1) * P.fplan.gate_rc.size() * 32;
            for (const ttn::FusedPass& ps : P.fplan.passes) {
                ttn_status s = launch_fcount_pass(&P, ps, st);
                if (s != TTN_OK) return s;
            }
        }
        cp.init = (c == 0); cp.reduce = (c == N - 1);
        cp.tables = reinterpret_cast<const float*>(base + cl.tables) + (size_t)c * Mp * 256;
        for (int r = 0; r < 8; ++r)
            for (int k = 0; k < 4; ++k)
                cp.jv[r][k] = (r >= 1 && r < M) ? -2.f * Jv[((size_t)(r - 1) * N + c) * 4 + k] : 0.f;
        ttn::chimera_column_count_kernel<<<cgrid, ttn::CH2C_WARPS * 32, 0, st>>>(cp);
        TTN_CUDA(cudaGetLastError());
    }
    ttn::final_reduce_kernel<true><<<1, 256, 0, st>>>(cp.part_x, cp.part_n, (unsigned long long)cgrid,
                                                     reinterpret_cast<float*>(base + cl.lay.out_x), reinterpret_cast<double*>(base + cl.lay.out_n));
    TTN_CUDA(cudaGetLastError());
    float mx = 0; double g = 0;
    TTN_CUDA(cudaMemcpyAsync(&mx, base + cl.lay.out_x, sizeof(float), cudaMemcpyDeviceToHost, st));
    TTN_CUDA(cudaMemcpyAsync(&g, base + cl.lay.out_n, sizeof(double), cudaMemcpyDeviceToHost, st));
    TTN_CUDA(cudaStreamSynchronize(st));
    const double top = (double)mx + shift;
    *E0 = top == 0.0 ? 0.0 : -top;
    *degeneracy = g;                                         // (the padded cells' free spins were divided out per column)
    return TTN_OK;
}

// ---- ttn_sweep_energy_noalloc: the energy sweep for callers that have no device memory to give -------
//
// Every other compute call of this library works inside a device workspace the caller allocates.  Some
// callers cannot do that: a plug-in or callback living inside a host application that has already given
// the whole GPU to its own memory pool (a raw cudaMalloc there fails, and the plug-in holds no handle to
// the pool), or a loop that must never meet the device-wide synchronisation cudaMalloc / cudaFree imply.
// For them the workspace of this one call is the array below: it is part of the library image, so every
// GPU that loads libttn.so holds TTN_NOALLOC_SCRATCH_BYTES of it from load until the process exits.
//
// On the host, `g_noalloc_scratch` is only a handle for the runtime's symbol table, NOT a device address:
// handing it to a kernel would fault (or, where the GPU can reach host memory, quietly use the wrong
// bytes).  The device address is looked up with cudaGetSymbolAddress, once per device, with that device
// current, by the first call made on it -- that first call should therefore happen outside any stream
// capture.  The kernels then receive that address exactly like a caller's workspace pointer.
static __device__ __align__(256) unsigned char g_noalloc_scratch[TTN_NOALLOC_SCRATCH_BYTES];

namespace {
constexpr int NOALLOC_MAX_DEVICES = 64;
void* g_noalloc_addr[NOALLOC_MAX_DEVICES] = {};      // per device ordinal: device address of the array
std::mutex g_noalloc_mu;

ttn_status noalloc_scratch(void** out) {
    int dev = -1;
    TTN_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= NOALLOC_MAX_DEVICES) return fail(TTN_EUNSUPPORTED, "device ordinal %d beyond %d", dev, NOALLOC_MAX_DEVICES);
    std::lock_guard<std::mutex> lock(g_noalloc_mu);
    if (!g_noalloc_addr[dev]) {
        void* p = nullptr;
        TTN_CUDA(cudaGetSymbolAddress(&p, g_noalloc_scratch));     // the copy of the array on the current device
        if (!p || (uintptr_t)p % 256) return fail(TTN_ECUDA, "cudaGetSymbolAddress gave an unusable address %p", p);
        g_noalloc_addr[dev] = p;
    }
    *out = g_noalloc_addr[dev];
    return TTN_OK;
}
}  // namespace

extern "C" ttn_status ttn_sweep_energy_noalloc(int L, const float* Jh, const float* Jv, const float* h, int batch,
                                               void* stream, double* E0) {
    if (!E0) return fail(TTN_EINVAL, "E0 is NULL");
    if (L < 1 || batch < 1) return fail(TTN_EINVAL, "L and batch must be >= 1");
    if (L > 1 && (!Jh || !Jv)) return fail(TTN_EINVAL, "Jh/Jv is NULL");
    // the size the ordinary call would ask its caller for (the smaller half-state size when there is no field)
    bool field = false;
    if (h) for (size_t i = 0, n = (size_t)batch * L * L; i < n && !field; ++i) field = (h[i] != 0.0f);
    const size_t need = field ? ttn_workspace_bytes(2, L, TTN_TROPICAL_F32, batch, 0)
                              : ttn_workspace_bytes_h0(2, L, TTN_TROPICAL_F32, batch, 0);
    if (need == 0) return fail(TTN_EUNSUPPORTED, "L=%d beyond the limits for this call", L);
    if (need > (size_t)TTN_NOALLOC_SCRATCH_BYTES)
        return fail(TTN_EUNSUPPORTED, "ttn_sweep_energy_noalloc: L=%d, batch=%d needs %zu bytes of scratch, the built-in array holds %zu "
                    "(L <= 20 with a field, L <= 21 without, batch 1); use ttn_sweep_energy with a workspace of your own",
                    L, batch, need, (size_t)TTN_NOALLOC_SCRATCH_BYTES);
    void* scratch = nullptr;
    ttn_status s = noalloc_scratch(&scratch);
    if (s != TTN_OK) return s;
    // Nothing in the array has to start at zero: the first pass of a sweep writes every state element without
    // reading it, the tables are uploaded or computed by the prep kernel, and every partial is written before the
    // final reduction reads it -- so what the previous call left behind is never read.
    return one_call(2, L, TTN_CALL_ENERGY, Jh, Jv, h, batch, scratch, (size_t)TTN_NOALLOC_SCRATCH_BYTES, stream, E0, nullptr, nullptr);
}
