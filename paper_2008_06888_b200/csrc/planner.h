// planner.h -- host-side pass scheduler for the tropical transfer sweep.
//
// The circuit of Fig. 1(b) has three kinds of operation on the q^L state:
//   g(r,c)   r >= 1 : the single-site max-plus gate (A2) PAPER.md:242 carrying Jv[r-1][c]
//                     (couples row r-1 to row r) on digit c;
//   dh(r,c)         : the field gate (A3) PAPER.md:247, diagonal:  += h[r][c] * sigma_c;
//   dJ(r,c) c < L-1 : the two-site diagonal gate (A4) PAPER.md:251: += Jh[r][c] sigma_c sigma_c+1.
// "The order of operation of these diagonal gates ... can be arbitrary"; gates on
// different digits commute.  Two operations fail to commute only when one is a gate on digit c
// and the other is a gate on c or a diagonal that reads digit c:
//     g(r,c)  before  dh(r,c), dJ(r,c-1), dJ(r,c)  before  g(r+1,c).
// Both kernel paths run in the DIAGONAL FRAME (defined at the fused section below): all dh / dJ
// are folded into conjugated gates, and the rule becomes the three-point stencil
//     g(r,c)  after  g(r-1,c-1), g(r-1,c), g(r-1,c+1);   gates of one row commute.
// A pass holds a set of digits in its tile (a contiguous low block [0,lo) that "rides" for
// coalescing plus a high block [a,b)) and may apply any legal gate whose digit is in the tile.
// The planner visits a cyclic sequence of overlapping tiles and, in each pass, greedily applies
// every gate that has become legal -- trapezoids/parallelograms over (row, column) as deep as
// the tile allows -- which cuts HBM passes from ceil(L/T) per row to well below one.
//
// Host only; no CUDA.  The same structures are dumped by ttn_plan_describe() and replayed by
// tests/test_planner.py against an independent statement of the rule.
#pragma once
#include <algorithm>
#include <cstdint>
#include <cstdio>
#include <string>
#include <vector>

namespace ttn {

enum OpType : uint8_t { OP_GATE = 0 };     // diagonal frame: gates are the only scheduled operation

struct Op {            // 8 bytes, uploaded as-is
    uint8_t type;      // OpType
    uint8_t pos;       // GATE: tile position of the digit (0 .. T-1)
    uint8_t c;         // global column (digit)
    uint8_t first;     // 1 = first gate of a round (the gates of a round commute: all were legal together)
    uint16_t row;      // lattice row r of the operation
    uint16_t nb;       // q = 3 (mark_gate_blocks): this gate leads a block of nb gates on adjacent columns
                       // of one row, applied together; 0 = member of the preceding block.  1 otherwise.
};

enum PassFlags : int { PASS_INIT = 1, PASS_REDUCE = 2 };

struct Pass {
    int lo, a, b;          // tile digits = [0,lo) U [a,b), a >= lo; T = lo + (b-a)
    int op_begin, op_end;  // into Plan::ops
    int flags;
    int src_buf, dst_buf;  // -1 = the state V; r >= 0 = checkpoint C_r
    int n_gates;
};

// COLOUR-ROTATION (Z3) REDUCTION of the Potts sweep (q = 3; there are no fields, App. C).
// E = -sum J delta(t_i, t_j) is invariant under t -> t + 1 (mod 3) on every site, every 3 x 3 gate and
// every diagonal commutes with that rotation rho, and the initial state is rho-invariant: every
// intermediate state obeys W[t] = W[rho t].  Only the third with column 0 in colour 0 is stored: a state
// over the L - 1 digits of columns 1 .. L-1 (digit d = column d + 1).  Gates on columns >= 1 stay inside
// it (column 1's left neighbour is the constant colour 0).  The gate on column 0 acts on the triple
// W[k, rest] = H[rho^-k rest], k = 0, 1, 2: three stored elements whose EVERY digit differs by the same
// shift -- they live in the three tiles of a rotation orbit, which one CTA holds together.  That
// "virtual column" gate (Op.c = Op.pos = VCOL) touches no tile digit and is legal in any pass; by the
// three-point stencil it depends on column 1 (digit 0).  Plan::vcol: L counts the stored DIGITS, the
// lattice has L + 1 rows.
constexpr int VCOL = 255;

struct Plan {
    int q = 2, L = 0;
    bool vcol = false;          // Z3-reduced Potts plan (see above)
    bool row_aligned = false;   // ttn_ground_config: every row boundary is materialised
    std::vector<Pass> passes;
    std::vector<Op> ops;
};

struct TileSpec { int lo, a, b; };

// Generic-path scheduler in the DIAGONAL FRAME (see the fused section below for the frame): only
// gates are scheduled; g(r,c) is legal once g(r-1,c-1), g(r-1,c), g(r-1,c+1) are done.
class Scheduler {
  public:
    explicit Scheduler(int L, bool vcol = false) : L_(L), rows_(vcol ? L + 1 : L), vcol_(vcol), grow_(L, 1) {}
    bool done() const {
        for (int c = 0; c < L_; ++c) if (grow_[c] != rows_) return false;
        return !vcol_ || vgrow_ == rows_;
    }
    bool row_done(int r) const {   // all of row r's gates applied
        for (int c = 0; c < L_; ++c) if (grow_[c] < r + 1) return false;
        return !vcol_ || vgrow_ >= r + 1;
    }
    // Greedily apply everything legal for tile digits [0,lo) U [a,b) with rows <= max_row.
    // Appends to ops; returns number of gates applied.
    int run_pass(const TileSpec& t, int max_row, std::vector<Op>& ops) {
        int gates = 0;
        auto in_tile = [&](int c) { return c < t.lo || (c >= t.a && c < t.b); };
        auto pos_of = [&](int c) { return c < t.lo ? c : t.lo + (c - t.a); };
        for (;;) {
            std::vector<int> legal;                          // legal at the start of this round
            for (int c = 0; c < L_; ++c) {
                if (!in_tile(c)) continue;
                const int r = grow_[c];
                if (r >= rows_ || r > max_row) continue;
                if (c > 0 && grow_[c - 1] < r) continue;
                if (c == 0 && vcol_ && vgrow_ < r) continue;     // digit 0 = column 1: its left neighbour is column 0
                if (c + 1 < L_ && grow_[c + 1] < r) continue;
                legal.push_back(c);
            }
            // the virtual column 0: in every tile; its only neighbour is digit 0 (column 1)
            const bool vlegal = vcol_ && vgrow_ < rows_ && vgrow_ <= max_row && grow_[0] >= vgrow_;
            if (legal.empty() && !vlegal) break;
            bool first = true;
            for (int c : legal) {
                ops.push_back({OP_GATE, (uint8_t)pos_of(c), (uint8_t)c, (uint8_t)(first ? 1 : 0), (uint16_t)grow_[c], 1});
                first = false;
                ++gates;
            }
            if (vlegal) { ops.push_back({OP_GATE, (uint8_t)VCOL, (uint8_t)VCOL, (uint8_t)(first ? 1 : 0), (uint16_t)vgrow_, 1}); ++gates; }
            for (int c : legal) grow_[c] += 1;
            if (vlegal) vgrow_ += 1;
        }
        return gates;
    }
  private:
    int L_, rows_;
    bool vcol_;
    int vgrow_ = 1;                    // rows complete on the virtual column
    std::vector<int> grow_;            // grow[c] = rows complete on digit c (row 0 needs no gate)
};

// Tile cycle: first tile [0, w0) (contiguous), then high tiles of `wh` active digits with
// `ride` low riding digits, starts advancing by `stride`, the last one flush with digit L.
inline std::vector<TileSpec> tile_cycle(int L, int Tmax, int ride, int stride) {
    std::vector<TileSpec> t;
    int w0 = Tmax < L ? Tmax : L;
    t.push_back({w0, w0, w0});
    if (w0 == L) return t;
    int wh = Tmax - ride;
    int x = w0 - (wh - stride);
    for (;;) {
        if (x + wh >= L) x = L - wh;
        if (x < ride) t.push_back({x + wh, x + wh, x + wh});   // degenerate: still a low tile
        else t.push_back({ride, x, x + wh});
        if (x + wh >= L) break;
        x += stride;
    }
    return t;
}

// Build the plan.  Tmax = log_q of the tile capacity; ride = riding low digits of high tiles.
inline Plan make_plan(int q, int L, bool has_field, bool row_aligned, int Tmax, int ride, bool vcol = false) {
    Plan best;
    int wh = Tmax - ride;
    int s_lo = 1, s_hi = wh;
    if (Tmax >= L) { s_lo = s_hi = 1; }
    if (row_aligned) { s_lo = s_hi = wh; }
    bool have = false;
    for (int stride = s_lo; stride <= s_hi; ++stride) {
        std::vector<TileSpec> cyc = tile_cycle(L, Tmax, ride, stride);
        Plan p; p.q = q; p.L = L; p.row_aligned = row_aligned; p.vcol = vcol;
        Scheduler s(L, vcol);
        size_t k = 0; int row = 0; bool first = true; int idle = 0;
        int cur_src = -1;
        while (first || !s.done()) {   // the INIT pass exists even when there is nothing to apply
            const TileSpec& t = cyc[k % cyc.size()]; ++k;
            Pass ps{t.lo, t.a, t.b, (int)p.ops.size(), 0, 0, -1, -1, 0};
            ps.n_gates = s.run_pass(t, row_aligned ? row : L + 1, p.ops);
            ps.op_end = (int)p.ops.size();
            if (ps.op_end == ps.op_begin && !first) { if (++idle > (int)cyc.size()) break; continue; }
            idle = 0;
            if (first) ps.flags |= PASS_INIT;
            first = false;
            if (row_aligned) {
                ps.src_buf = cur_src;
                if (s.row_done(row)) { ps.dst_buf = row; cur_src = row; ++row; k = 0; }
                else { ps.dst_buf = -1; cur_src = -1; }
            }
            p.passes.push_back(ps);
        }
        if (!s.done()) continue;
        if (!row_aligned && !p.passes.empty()) p.passes.back().flags |= PASS_REDUCE;
        if (!have || p.passes.size() < best.passes.size()) { best = p; have = true; }
    }
    return best;
}

// Beam search over tile sequences (any tile at any step instead of a fixed cycle): minimises the
// number of HBM passes of a multi-pass sweep; among sequences of equal length the one with more
// low (contiguous) tiles wins, since a strided pass costs about twice the memory time of a
// contiguous one (profiles/r01j.md).  States are the per-column progress vectors; a layer holds
// the `width` states with the most gates applied.  Used for the q = 3 plans, where a pass costs
// 15-20 ms of memory time before its first gate.
inline Plan make_plan_beam(int q, int L, int Tmax, int ride, int width = 256, bool vcol = false) {
    const int wh = Tmax - ride;
    const int rows = vcol ? L + 1 : L;          // progress vectors carry the virtual column at index L
    std::vector<TileSpec> tiles;
    tiles.push_back({Tmax, Tmax, Tmax});
    for (int a = ride + 1; a + wh <= L; ++a) tiles.push_back({ride, a, a + wh});
    struct Node { std::vector<int> grow; std::vector<int> seq; int total; int lows; };
    auto advance = [&](const std::vector<int>& g0, const TileSpec& t, std::vector<int>& g1) {
        g1 = g0;
        int gates = 0;
        auto in_tile = [&](int c) { return c < t.lo || (c >= t.a && c < t.b); };
        for (;;) {
            int legal[64], nl = 0;
            for (int c = 0; c < L; ++c) {
                if (!in_tile(c)) continue;
                const int r = g1[c];
                if (r >= rows) continue;
                if (c > 0 && g1[c - 1] < r) continue;
                if (c == 0 && vcol && g1[L] < r) continue;
                if (c + 1 < L && g1[c + 1] < r) continue;
                legal[nl++] = c;
            }
            const bool vlegal = vcol && g1[L] < rows && g1[0] >= g1[L];
            if (!nl && !vlegal) break;
            for (int i = 0; i < nl; ++i) g1[legal[i]] += 1;
            if (vlegal) g1[L] += 1;
            gates += nl + (vlegal ? 1 : 0);
        }
        return gates;
    };
    const int all_gates = vcol ? (L + 1) * L : L * (L - 1);
    std::vector<Node> layer(1);
    layer[0].grow.assign(vcol ? L + 1 : L, 1); layer[0].total = 0; layer[0].lows = 0;
    std::vector<int> best_seq;
    for (int depth = 0; depth < 4 * L && best_seq.empty(); ++depth) {
        std::vector<Node> next;
        for (const Node& nd : layer)
            for (size_t ti = 0; ti < tiles.size(); ++ti) {
                Node nn;
                const int g = advance(nd.grow, tiles[ti], nn.grow);
                if (g == 0 && depth > 0) continue;
                nn.seq = nd.seq; nn.seq.push_back((int)ti);
                nn.total = nd.total + g; nn.lows = nd.lows + (ti == 0);
                next.push_back(std::move(nn));
            }
        if (next.empty()) break;
        // best first: most gates applied, then most low tiles; drop duplicates of a progress vector
        std::stable_sort(next.begin(), next.end(), [](const Node& x, const Node& y) {
            if (x.total != y.total) return x.total > y.total;
            return x.lows > y.lows;
        });
        layer.clear();
        for (Node& nn : next) {
            bool dup = false;
            for (const Node& k : layer) if (k.grow == nn.grow) { dup = true; break; }
            if (dup) continue;
            if (nn.total == all_gates) { if (best_seq.empty()) best_seq = nn.seq; continue; }
            if ((int)layer.size() < width) layer.push_back(std::move(nn));
        }
    }
    Plan p; p.q = q; p.L = L; p.row_aligned = false; p.vcol = vcol;
    if (best_seq.empty()) return p;
    Scheduler s(L, vcol);
    for (size_t i = 0; i < best_seq.size(); ++i) {
        const TileSpec& t = tiles[best_seq[i]];
        Pass ps{t.lo, t.a, t.b, (int)p.ops.size(), 0, 0, -1, -1, 0};
        ps.n_gates = s.run_pass(t, L + 1, p.ops);
        ps.op_end = (int)p.ops.size();
        if (i == 0) ps.flags |= PASS_INIT;
        p.passes.push_back(ps);
    }
    if (!s.done()) { p.passes.clear(); p.ops.clear(); return p; }
    p.passes.back().flags |= PASS_REDUCE;
    return p;
}

// q = 3 (ttn_potts.cuh): group the gates of every round into blocks of up to max_nb gates on
// adjacent columns held at adjacent tile positions.  Gates legal in the same round on adjacent
// columns belong to the same lattice row (each needs its neighbour to be at least as far), so a
// block shares one conjugation A_{r-1}.  Runs are cut 3,3,..., with a tail of 2+2 instead of 3+1.
inline void mark_gate_blocks(Plan& p, int max_nb = 3) {
    for (const Pass& ps : p.passes) {
        int k = ps.op_begin;
        while (k < ps.op_end) {
            int run = 1;
            while (k + run < ps.op_end && !p.ops[k + run].first && p.ops[k + run].row == p.ops[k].row &&
                   p.ops[k + run].c == p.ops[k + run - 1].c + 1 && p.ops[k + run].pos == p.ops[k + run - 1].pos + 1)
                ++run;
            int left = run, i = k;
            while (left > 0) {
                int nb = left < max_nb ? left : max_nb;
                if (max_nb == 3 && left == 4) nb = 2;
                p.ops[i].nb = (uint16_t)nb;
                for (int j = 1; j < nb; ++j) p.ops[i + j].nb = 0;
                i += nb; left -= nb;
            }
            k += run;
        }
    }
}

inline std::string describe(const Plan& p) {
    std::string out;
    char line[160];
    snprintf(line, sizeof line, "plan q=%d L=%d row_aligned=%d passes=%zu ops=%zu vcol=%d\n", p.q, p.L,
             (int)p.row_aligned, p.passes.size(), p.ops.size(), (int)p.vcol);
    out += line;
    for (size_t i = 0; i < p.passes.size(); ++i) {
        const Pass& ps = p.passes[i];
        snprintf(line, sizeof line, "pass %zu lo=%d a=%d b=%d flags=%d src=%d dst=%d gates=%d nops=%d\n",
                 i, ps.lo, ps.a, ps.b, ps.flags, ps.src_buf, ps.dst_buf, ps.n_gates, ps.op_end - ps.op_begin);
        out += line;
        for (int k = ps.op_begin; k < ps.op_end; ++k) {
            const Op& o = p.ops[k];
            snprintf(line, sizeof line, "op %s r=%d c=%d pos=%d first=%d nb=%d\n",
                     "g", o.row, o.c, o.pos, o.first, o.nb);
            out += line;
        }
    }
    return out;
}


// =============================================================================================
// Fused register-phase schedule in the DIAGONAL FRAME ("v3", Ising Tropical<f32>).
//
// Diagonal frame.  Let D_r be the product of all diagonal gates of row r ((A3), (A4)
// PAPER.md:247-252) and A_r = D_0 D_1 ... D_r (diagonal operators commute).  With
// G_r(c) the max-plus gate (A2) PAPER.md:242 of row r on digit c, the sweep
//     V = D_{L-1} G_{L-1} ... D_1 G_1 D_0 1         equals        V = A_{L-1} G''_{L-1} ... G''_1 1,
//     G''_r(c) = A_{r-1}^{-1} G_r(c) A_{r-1}        (a similarity transform of every gate).
// A_{r-1}(s) = sum_c H_c sigma_c + sum_c K_c sigma_c sigma_{c+1} with H_c = sum_{r'<r} h[r'][c],
// K_c = sum_{r'<r} Jh[r'][c], so G''_r(c) is still a 2x2 max-plus gate on digit c, whose two
// off-diagonal entries depend on the neighbour bits c-1 and c+1 of the element's own index:
//     a' = max(a, b + m - 2 rho),  b' = max(b, a + m + 2 rho),   m = -2 Jv[r-1][c],
//     rho = H_c + K_{c-1} sigma_{c-1} + K_c sigma_{c+1}          (8 constants per gate).
// No diagonal pass over the state is ever made; the last pass adds A_{L-1}(s) before the final
// (+)-reduction.  Dependency rule in this frame: g''(r,c) needs g''(r-1,c-1), g''(r-1,c),
// g''(r-1,c+1); gates of one row commute with each other (same conjugation), gates on
// non-adjacent digits always commute.
//
// Every WARP owns a tile of 2^12 state elements, 128 per thread (7 "register digits"):
//   LOW  tile (a = 0): 12 active digits d0..d11 = columns 0..11, a contiguous 16 KiB chunk.
//        layout A: register digits d0..d6, lane digits d7..d11
//        layout B: register digits d5..d11, lane digits d0..d4     (loads/stores: 128 B coalesced)
//   HIGH tile (a >= 4): 9 active digits d0..d8 = columns a..a+8 plus the 3 riding digits 0..2,
//        which sit on the low 3 lane bits so that every global request moves whole 32-byte runs.
//        layout A: register digits d0..d6, lanes (riding, d7, d8)
//        layout B: register digits d2..d8, lanes (riding, d0, d1)
// A gate on a register digit is pure register arithmetic; its neighbour bits are register-index
// bits (compile-time per unrolled element) or constant per thread (lane / tile bits).
// MIRRORED LAYOUTS.  The 7 register digits form a chain p0..p6; in layout A p_i is the i-th
// register digit from the LEFT, in layout B the i-th from the RIGHT.  Chain positions sit on the
// same register-index bits in both layouts, so one set of 7 unrolled gate bodies serves both
// (the instruction footprint is what the SM's instruction cache has to hold): the body of bit K
// only knows its "P" neighbour (chain position - 1; the tile's outer neighbour column for p0)
// and its "Q" neighbour (position + 1; a lane digit for p6).  P/Q are left/right in A and
// right/left in B; the gate constants are stored as k[side][P bit][Q bit].
// A phase is a list of ROUNDS; a round applies, for a 7-bit mask of register bits, the next gate
// of each of those digits (all legal at the start of the round), in ascending bit order.  Layout
// exchanges go through the warp's private shared-memory region.
// =============================================================================================
enum MicroCode : uint8_t { MC_END = 0, MC_XAB = 1, MC_XBA = 2, MC_ROUND = 3, MC_FINAL = 4,
                            MC_CKPT = 5 };   // store the tile as it stands to the pass's checkpoint buffer (merged row plans)

struct MicroOp { uint8_t code; uint8_t mask; uint16_t arg; };   // ROUND: mask = register bits, arg = index of
                                                                // its first gate in the pass's gate list
                                                                // | MOP_FLIP: the round ends with the Z2 flip gate
constexpr uint16_t MOP_FLIP = 0x8000;       // (column 0, see "GLOBAL-FLIP (Z2) REDUCTION" below)
constexpr int GATE_RC_FLIP = 1 << 17;       // gate_rc flag of a flip gate (its K field is 0)

constexpr int F_RB = 7;          // register digits
constexpr int F_WLOW = 12;       // active digits of the low tile
constexpr int F_WHIGH = 9;       // active digits of a high tile
constexpr int F_RIDE = 3;        // riding digits of a high tile
constexpr int F_AMIN = 4;        // smallest start of a high tile (its outer neighbour must not ride)

// tile digit (0..W-1) held by register-index bit `bit` in `layout` of a low/high tile
//   lowA {5,6,0,1,2,3,4}   lowB {6,5,11,10,9,8,7}   highA {4,5,6,0,1,2,3}   highB {4,3,2,8,7,6,5}
// chain position of a bit = its layout-A digit; layout B holds digit (W-1) - position.
#if defined(__CUDACC__)
__host__ __device__
#endif
constexpr int fused_chain_pos(bool low, int bit) {
    return low ? (bit < 2 ? 5 + bit : bit - 2) : (bit < 3 ? 4 + bit : bit - 3);
}
#if defined(__CUDACC__)
__host__ __device__
#endif
constexpr int fused_digit_of_bit(bool low, int layout, int bit) {
    return layout == 0 ? fused_chain_pos(low, bit) : (low ? 11 : 8) - fused_chain_pos(low, bit);
}
// register-index bit holding tile digit d in this layout, or -1 (lane / tile digit)
#if defined(__CUDACC__)
__host__ __device__
#endif
constexpr int fused_bit_of_digit(bool low, int layout, int d) {
    for (int b = 0; b < F_RB; ++b) if (fused_digit_of_bit(low, layout, b) == d) return b;
    return -1;
}

// Tile geometry of a fused kernel family.
//  kind 0: Tropical<f32>, 128 elements per thread (7 register digits, maps above).
//  kind 1: CountingTropical<f32,f64>, 32 elements per thread (5 register digits; a tile is 2^10
//          elements: LOW = columns 0..9, HIGH = 3 riding + 7 active); register bit i holds chain
//          position i: digit i in layout A, digit W-1-i in layout B.
//  kind 2: Tropical<i16>, two elements per 32-bit word: column 0 is the HALF of a word and the
//          kind-0 geometry applies to the word index (column c >= 1 = word digit c-1).  The LOW
//          tile has 13 columns; pseudo register bit 7 is the half digit (in every LOW layout);
//          HIGH tiles start at column a >= 5 (word digit a-1) and column 0 rides.
//
// GLOBAL-FLIP (Z2) REDUCTION, h = 0 (symmetry of Eq. (1) PAPER.md:29 without the
// field term).  Every gate (A2) and every diagonal (A4) commutes with the flip F: s -> ~s, and the
// initial state is F-invariant, so EVERY intermediate state of every schedule obeys W[s] = W[~s].
// Only the half with column 0 up (s_0 = 0) is stored: an (L-1)-digit state u = (s_1 .. s_{L-1}).
//   * a gate on column c >= 1 stays inside the half; column 1's left neighbour is the constant
//     sigma_0 = +1 (the kernels' "column -1 does not exist" bit 0, with K_0 in the constants);
//   * the gate on column 0 pairs s with the element whose column-0 bit is set, which the symmetry
//     maps to the COMPLEMENT of u inside the half:
//         W'[u] = max(W[u], W[~u] + m - 2 K_0 sigma_1(u)),    m = -2 Jv[r-1][0];
//     it touches no particular digit, so it is legal in any tile; it depends, by the usual
//     stencil, on column 1, which the LOW tile holds: it is scheduled there as pseudo register
//     bit RB (+1) of every LOW layout, and the LOW kernel pairs warps on tiles (T, ~T).
//  kind 3: Tropical<f32> + Z2: the kind-0 geometry on the digits d = c - 1 (same column maps as kind 2)
//  kind 4: CountingTropical + Z2: the kind-1 geometry on d = c - 1, pseudo bit 5 = column 0
//  kind 5: Tropical<i16> + Z2: column 1 is the half of a word (pseudo bit 7), word digit = c - 2,
//          pseudo bit 8 = column 0
struct FusedGeom { int RB, WLOW, WHIGH, RIDE, AMIN, kind; };
constexpr FusedGeom GEOM_F32{F_RB, F_WLOW, F_WHIGH, F_RIDE, F_AMIN, 0};
constexpr FusedGeom GEOM_COUNT{5, 10, 7, 3, 4, 1};
constexpr FusedGeom GEOM_I16{F_RB, F_WLOW + 1, F_WHIGH, F_RIDE + 1, F_AMIN + 1, 2};
constexpr FusedGeom GEOM_F32_Z2{F_RB, F_WLOW + 1, F_WHIGH, F_RIDE + 1, F_AMIN + 1, 3};
constexpr FusedGeom GEOM_COUNT_Z2{5, 11, 7, 4, 5, 4};
constexpr FusedGeom GEOM_I16_Z2{F_RB, F_WLOW + 2, F_WHIGH, F_RIDE + 2, F_AMIN + 2, 5};
// columns in front of the first tile digit of the kernel's index space (virtual / sub-word columns)
#if defined(__CUDACC__)
__host__ __device__
#endif
constexpr int geom_col_off(const FusedGeom& g) { return g.kind == 2 || g.kind == 3 || g.kind == 4 ? 1 : (g.kind == 5 ? 2 : 0); }
#if defined(__CUDACC__)
__host__ __device__
#endif
constexpr bool geom_has_flip(const FusedGeom& g) { return g.kind >= 3; }
// bits of a ROUND mask: the register bits, + the half-of-a-word column of the i16 LOW tiles (bit RB)
#if defined(__CUDACC__)
__host__ __device__
#endif
constexpr int geom_bits(const FusedGeom& g, bool low) { return (g.kind == 2 || g.kind == 5) && low ? g.RB + 1 : g.RB; }
// lattice column (relative to the tile start a; LOW tiles: a = 0) acted on by mask bit `bit`
#if defined(__CUDACC__)
__host__ __device__
#endif
constexpr int geom_digit_of_bit(const FusedGeom& g, bool low, int layout, int bit) {
    if (g.kind == 0) return fused_digit_of_bit(low, layout, bit);
    if (g.kind == 1) return layout == 0 ? bit : (low ? g.WLOW : g.WHIGH) - 1 - bit;
    if (g.kind == 4) return low ? 1 + (layout == 0 ? bit : g.WLOW - 2 - bit) : (layout == 0 ? bit : g.WHIGH - 1 - bit);
    if (!low) return fused_digit_of_bit(false, layout, bit);
    if (g.kind == 5) return bit == F_RB ? 1 : 2 + fused_digit_of_bit(true, layout, bit);
    if (g.kind == 3) return 1 + fused_digit_of_bit(true, layout, bit);
    return bit == F_RB ? 0 : 1 + fused_digit_of_bit(true, layout, bit);       // kind 2
}

struct FusedPass {
    int a, W;                    // active digits [a, a+W)
    int low;                     // 1 = low tile
    int flags;
    int first_layout, last_layout;
    int mop_begin, mop_end;      // into FusedPlan::mops
    int gate_begin, gate_end;    // into FusedPlan::gate_rc
    int n_phases, n_rounds;
    int src_buf = -1, dst_buf = -1;   // -1 = the state V; r >= 0 = checkpoint C_r (row-aligned plans)
    int ckpt_buf = -1;                // merged row plans: the row whose checkpoint the MC_CKPT micro-op of this pass writes
};

struct FusedPlan {
    int L = 0;
    std::vector<FusedPass> passes;
    std::vector<MicroOp> mops;
    std::vector<int> gate_rc;    // low << 16 | register bit << 13 | layout << 12 | r << 6 | c, in execution order
    bool ok = false;
};

class FusedScheduler {
  public:
    FusedScheduler(int L, FusedPlan& p, const FusedGeom& g = GEOM_F32) : L_(L), Pp_(&p), G_(g), grow_(L, 1) {}
    void rebind(FusedPlan& p) { Pp_ = &p; }
    bool done() const {
        for (int c = 0; c < L_; ++c) if (grow_[c] != L_) return false;
        return true;
    }
    // One pass over active digits [a, a+W).  Returns number of gates applied.
    bool row_done(int r) const {
        for (int c = 0; c < L_; ++c) if (grow_[c] < r + 1) return false;
        return true;
    }
    void set_max_row(int r) { max_row_ = r; }
    // gate-row plans: the gates of the current row on columns >= c are someone else's: count them as done
    void skip_columns_from(int c) { for (int i = c; i < L_; ++i) grow_[i] += 1; }
    // ckpt_row >= 0 (merged row plans): gates up to row ckpt_row, MC_CKPT (row ckpt_row is complete there: the
    // caller guarantees it), then the tile's gates of row ckpt_row + 1.
    int run_pass(int a, bool low, int max_gates, FusedPass& ps, int ckpt_row = -1) {
        if (ckpt_row >= 0) max_row_ = ckpt_row;
        const int W = low ? G_.WLOW : G_.WHIGH;
        ps.a = a; ps.W = W; ps.low = low; ps.flags = 0; ps.n_phases = 0; ps.n_rounds = 0;
        ps.mop_begin = (int)Pp_->mops.size(); ps.gate_begin = (int)Pp_->gate_rc.size();
        pass_gate_begin_ = ps.gate_begin; pass_mop_begin_ = ps.mop_begin; max_gates_ = max_gates;
        // the low tile loads and stores in layout B (coalesced); high tiles start in A
        int layout = low ? 1 : 0;
        ps.first_layout = layout;
        int total = 0, idle = 0;
        bool pending_x = false;                        // an exchange is owed before the next non-empty phase
        int cur = layout;                              // the layout the registers are in
        for (int part = 0; part < (ckpt_row >= 0 ? 2 : 1); ++part) {
            idle = 0;
            while (idle < 2) {
                size_t mark = Pp_->mops.size();
                if (pending_x) Pp_->mops.push_back({(uint8_t)(layout == 1 ? MC_XAB : MC_XBA), 0, 0});
                int rounds = 0;
                int n = run_phase(a, low, layout, rounds);
                if (n == 0) { Pp_->mops.resize(mark); ++idle; layout ^= 1; pending_x = !pending_x; continue; }
                total += n; idle = 0; ++ps.n_phases; ps.n_rounds += rounds;
                cur = layout;
                layout ^= 1; pending_x = true;
            }
            if (part == 0 && ckpt_row >= 0) {
                // back to "no exchange owed" relative to the layout the registers are in; LOW tiles store from B
                if (low && cur != 1) { Pp_->mops.push_back({MC_XAB, 0, 0}); cur = 1; }
                Pp_->mops.push_back({MC_CKPT, 0, 0});
                ps.ckpt_buf = ckpt_row;
                layout = cur; pending_x = false;
                max_row_ = ckpt_row + 1;
            }
        }
        int last = cur;                                 // the layout of the last productive phase
        if (ps.n_phases == 0) last = ps.first_layout;
        if (low && last != 1) { Pp_->mops.push_back({MC_XAB, 0, 0}); last = 1; }
        ps.last_layout = last;
        Pp_->mops.push_back({MC_END, 0, 0});
        ps.mop_end = (int)Pp_->mops.size(); ps.gate_end = (int)Pp_->gate_rc.size();
        return total;
    }
  private:
    bool legal(int c) const {
        const int r = grow_[c];
        if (r >= L_ || r > max_row_) return false;
        if (c > 0 && grow_[c - 1] < r) return false;
        if (c + 1 < L_ && grow_[c + 1] < r) return false;
        return true;
    }
    int run_phase(int a, bool low, int layout, int& rounds) {
        int n = 0;
        for (;;) {
            const int nb = geom_bits(G_, low);
            if ((int)Pp_->gate_rc.size() - pass_gate_begin_ + nb + 1 > max_gates_) break;
            if ((int)Pp_->mops.size() - pass_mop_begin_ + 8 > max_mops_) break;
            unsigned mask = 0;
            for (int b = 0; b < nb; ++b) if (legal(a + geom_digit_of_bit(G_, low, layout, b))) mask |= 1u << b;
            const bool flip = low && geom_has_flip(G_) && legal(0);      // Z2: the gate on column 0
            if (!mask && !flip) break;
            Pp_->mops.push_back({MC_ROUND, (uint8_t)mask, (uint16_t)(((int)Pp_->gate_rc.size() - pass_gate_begin_) | (flip ? MOP_FLIP : 0))});
            for (int b = 0; b < nb; ++b) if (mask >> b & 1) {
                const int c = a + geom_digit_of_bit(G_, low, layout, b);
                Pp_->gate_rc.push_back((low ? 1 << 16 : 0) | (b << 13) | (layout << 12) | (grow_[c] << 6) | c);
                ++n;
            }
            if (flip) { Pp_->gate_rc.push_back(GATE_RC_FLIP | (low ? 1 << 16 : 0) | (layout << 12) | (grow_[0] << 6) | 0); ++n; }
            for (int b = 0; b < nb; ++b) if (mask >> b & 1) grow_[a + geom_digit_of_bit(G_, low, layout, b)] += 1;
            if (flip) grow_[0] += 1;
            ++rounds;
        }
        return n;
    }
    int L_; FusedPlan* Pp_; FusedGeom G_;
    std::vector<int> grow_;      // grow[c] = rows complete on digit c (row 0 needs no gate)
    int pass_gate_begin_ = 0, pass_mop_begin_ = 0, max_gates_ = 1 << 30;
    int max_mops_ = 120;         // micro-ops per pass the kernel stages (FMAX_MOPS = 128)
    int max_row_ = 1 << 30;      // row-aligned plans: no gate of a later row
};

// Estimated time of one pass in ms on B200 (fit over the measured launch lists, profiles/r01f.md):
// 0.267 ms per gate (FMNMX floor 0.231), a fixed part for the memory phases that do not hide, round
// dispatch and exchanges; a pass cannot beat its memory time.
inline double fused_pass_cost(const FusedPass& ps, const FusedGeom& G = GEOM_F32) {
    const int g = ps.gate_end - ps.gate_begin, x = ps.n_phases > 1 ? ps.n_phases - 1 : 0;
    if (G.kind == 3 || G.kind == 4) {            // Z2: the kind-0 / kind-1 pass over half the elements
        FusedPass q = ps;
        return 0.5 * fused_pass_cost(q, G.kind == 3 ? GEOM_F32 : GEOM_COUNT);
    }
    if (G.kind == 5) { FusedPass q = ps; return 0.5 * fused_pass_cost(q, GEOM_I16); }
    if (G.kind == 2) {
        // Tropical<i16>: half the bytes and half the alu work per element; tiles whose 9 active
        // word digits reach past bit 18 (> 256 pages of 2 MiB) are bound by address translation
        if (ps.low) { const double t = 1.0 + 0.165 * g + 0.02 * ps.n_rounds + 0.25 * x; return t > 4.0 ? t : 4.0; }
        const double t = 2.9 + 0.115 * g + 0.06 * ps.n_rounds + 0.25 * x;
        return t > 5.0 ? t : 5.0;
    }
    if (ps.low) { const double t = 1.2 + 0.267 * g + 0.02 * ps.n_rounds + 0.25 * x; return t > 6.5 ? t : 6.5; }
    const double t = 3.5 + 0.267 * g + 0.08 * ps.n_rounds + 0.25 * x;
    return t > 9.0 ? t : 9.0;
}

// Two tile orders are tried and the cheaper plan (by fused_pass_cost) wins:
//  * cyclic: the low tile [0,12), then high tiles [x, x+9) advancing by `stride`, the last flush
//    with L, for every stride;
//  * greedy: at every step the tile (low, or high at any start) that applies the most gates.
inline FusedPlan make_fused_plan(int L, int max_gates_per_pass, const FusedGeom& G = GEOM_F32) {
    FusedPlan best;
    if (L < G.WLOW) return best;
    double best_cost = -1;
    auto finish = [&](FusedPlan& p) {
        // the last pass adds A_{L-1}(s) and reduces: MC_FINAL replaces its MC_END
        p.passes.back().flags |= PASS_REDUCE;
        p.mops.back().code = MC_FINAL;
        double cost = 0;
        for (auto& ps : p.passes) cost += fused_pass_cost(ps, G);
        if (best_cost < 0 || cost < best_cost) { best = p; best_cost = cost; best.ok = true; }
    };
    for (int stride = 1; stride <= G.WHIGH; ++stride) {
        std::vector<int> starts;
        starts.push_back(0);
        if (L > G.WLOW) {
            int x = G.WLOW - (G.WHIGH - stride);
            for (;;) {
                if (x + G.WHIGH >= L) x = L - G.WHIGH;
                if (x < G.AMIN) x = G.AMIN;
                starts.push_back(x);
                if (x + G.WHIGH >= L) break;
                x += stride;
            }
        }
        FusedPlan p; p.L = L;
        FusedScheduler s(L, p, G);
        size_t k = 0; int idle = 0; bool first = true;
        while ((first || !s.done()) && p.passes.size() < 4096) {
            int a = starts[k % starts.size()]; ++k;
            FusedPass ps{};
            size_t m0 = p.mops.size();
            int n = s.run_pass(a, a == 0, max_gates_per_pass, ps);
            if (n == 0 && !first) { p.mops.resize(m0); if (++idle > (int)starts.size()) break; continue; }
            idle = 0;
            if (first) ps.flags |= PASS_INIT;
            first = false;
            p.passes.push_back(ps);
        }
        if (!s.done()) continue;
        finish(p);
    }
    if (L > G.WLOW) {                               // greedy by gate count
        FusedPlan p; p.L = L;
        FusedScheduler s(L, p, G);
        bool first = true;
        while ((first || !s.done()) && p.passes.size() < 4096) {
            int best_a = -1, best_n = -1;
            for (int a = 0; a + G.WHIGH <= L; a = (a == 0 ? G.AMIN : a + 1)) {
                FusedScheduler trial = s;                       // dry run on a copy
                FusedPlan scratch; scratch.L = L;
                trial.rebind(scratch);
                FusedPass ps{};
                const int n = trial.run_pass(a, a == 0, max_gates_per_pass, ps);
                if (n > best_n) { best_a = a; best_n = n; }                      // ties: the lowest start
            }
            if (best_n <= 0 && !first) break;
            FusedPass ps{};
            s.run_pass(best_a, best_a == 0, max_gates_per_pass, ps);
            if (first) ps.flags |= PASS_INIT;
            first = false;
            p.passes.push_back(ps);
        }
        if (s.done()) finish(p);
    }
    return best;
}

// Row-aligned plan for ttn_ground_config (f32 geometry): every row boundary is materialised as a
// checkpoint C_r = V''_r.  Row r needs one pass per tile of a cover of the columns (the low tile
// and high tiles up to column L); the pass that completes row r writes C_r, the first pass of
// row r+1 reads it.  Pass 0 initialises C_0 (no gate: V''_0 is the tropical one everywhere).
// G = GEOM_F32, or GEOM_F32_Z2 for h = 0 (the checkpoints are then half-states).
inline FusedPlan make_fused_row_plan(int L, int max_gates_per_pass, const FusedGeom& G = GEOM_F32) {
    FusedPlan p; p.L = L;
    if (L < G.WLOW) return p;
    std::vector<int> starts{0};
    for (int x = G.WLOW; x < L; x += G.WHIGH) {
        int a = x + G.WHIGH <= L ? x : L - G.WHIGH;
        if (a < G.AMIN) a = G.AMIN;
        starts.push_back(a);
    }
    FusedScheduler s(L, p, G);
    {   // row 0: initialise
        s.set_max_row(0);
        FusedPass ps{};
        s.run_pass(0, true, max_gates_per_pass, ps);
        ps.flags |= PASS_INIT; ps.src_buf = -1; ps.dst_buf = 0;
        p.passes.push_back(ps);
    }
    for (int r = 1; r < L; ++r) {
        s.set_max_row(r);
        int src = r - 1;
        for (size_t k = 0; k < starts.size(); ++k) {
            FusedPass ps{};
            const size_t m0 = p.mops.size();
            const int n = s.run_pass(starts[k], starts[k] == 0, max_gates_per_pass, ps);
            const bool done = s.row_done(r);
            if (n == 0 && !(done && src >= 0)) { p.mops.resize(m0); continue; }
            ps.src_buf = src; ps.dst_buf = done ? r : -1;
            src = -1;
            p.passes.push_back(ps);
            if (done) break;
        }
        if (!s.row_done(r)) return p;          // ok stays false
    }
    p.ok = true;
    return p;
}

// ONE row of gates on every column of an L-column lattice (row 1 only; no INIT, no REDUCE pass): the
// single-spin gates of the chimera sweep's horizontal couplings (ttn_chimera2.cuh), which run on the
// Ising pass kernels.  One pass per tile of a column cover, all in place.
// Columns >= ncols get no gate (the caller applies them elsewhere); the tiles cover [0, ncols).
inline FusedPlan make_gate_row_plan(int L, int ncols, int max_gates_per_pass, const FusedGeom& G) {
    FusedPlan p; p.L = L;
    if (L < G.WLOW || ncols > L) return p;
    std::vector<int> starts{0};
    for (int x = G.WLOW; x < ncols; x += G.WHIGH) {
        int a = x + G.WHIGH <= ncols ? x : ncols - G.WHIGH;
        if (a < G.AMIN) a = G.AMIN;
        starts.push_back(a);
    }
    FusedScheduler s(L, p, G);
    s.set_max_row(1);
    s.skip_columns_from(ncols);
    for (size_t k = 0; k < starts.size(); ++k) {
        FusedPass ps{};
        const size_t m0 = p.mops.size();
        const int n = s.run_pass(starts[k], starts[k] == 0, max_gates_per_pass, ps);
        if (n == 0) { p.mops.resize(m0); continue; }
        p.passes.push_back(ps);
    }
    p.ok = s.row_done(1);
    return p;
}

// Merged row-aligned plan (two tile kinds: the low tile and ONE high tile, i.e. L <= WLOW + WHIGH): the tile
// order alternates from row to row -- low, high | high, low | low, high ... -- so that the second pass of row
// r and the first pass of row r + 1 use the same tile and merge into one pass with the checkpoint store of
// C_r in its middle (MC_CKPT): one load of the tile for two rows of its gates, L passes instead of 2L - 1.
// Gates of one row commute (planner.h header), so the order inside a row is free.
inline FusedPlan make_fused_row_plan_merged(int L, int max_gates_per_pass, const FusedGeom& G = GEOM_F32) {
    FusedPlan p; p.L = L;
    if (L <= G.WLOW || L > G.WLOW + G.WHIGH) return p;
    int ah = L - G.WHIGH;
    if (ah < G.AMIN) ah = G.AMIN;
    FusedScheduler s(L, p, G);
    {   // row 0: initialise C_0
        s.set_max_row(0);
        FusedPass ps{};
        s.run_pass(0, true, max_gates_per_pass, ps);
        ps.flags |= PASS_INIT; ps.src_buf = -1; ps.dst_buf = 0;
        p.passes.push_back(ps);
    }
    {   // first half of row 1 on the low tile
        s.set_max_row(1);
        FusedPass ps{};
        s.run_pass(0, true, max_gates_per_pass, ps);
        ps.src_buf = 0; ps.dst_buf = -1;
        p.passes.push_back(ps);
    }
    bool low = false;                          // tile of the next (merged) pass
    for (int r = 1; r < L; ++r, low = !low) {
        FusedPass ps{};
        if (r + 1 < L) {
            s.run_pass(low ? 0 : ah, low, max_gates_per_pass, ps, /*ckpt_row=*/r);
            ps.src_buf = -1; ps.dst_buf = -1;
        } else {                               // the last row: its second half completes it
            s.set_max_row(r);
            s.run_pass(low ? 0 : ah, low, max_gates_per_pass, ps);
            ps.src_buf = -1; ps.dst_buf = r;
        }
        p.passes.push_back(ps);
        if (!s.row_done(r)) return p;          // ok stays false
    }
    p.ok = s.done();
    return p;
}

inline std::string describe_fused(const FusedPlan& p) {
    std::string out; char line[200];
    snprintf(line, sizeof line, "fused L=%d passes=%zu mops=%zu gates=%zu\n", p.L,
             p.passes.size(), p.mops.size(), p.gate_rc.size());
    out += line;
    for (size_t i = 0; i < p.passes.size(); ++i) {
        const FusedPass& ps = p.passes[i];
        snprintf(line, sizeof line, "fpass %zu a=%d W=%d low=%d flags=%d first=%d last=%d phases=%d rounds=%d gates=%d src=%d dst=%d ckpt=%d\n", i,
                 ps.a, ps.W, ps.low, ps.flags, ps.first_layout, ps.last_layout, ps.n_phases, ps.n_rounds,
                 ps.gate_end - ps.gate_begin, ps.src_buf, ps.dst_buf, ps.ckpt_buf);
        out += line;
        for (int k = ps.mop_begin; k < ps.mop_end; ++k) {
            const MicroOp& m = p.mops[k];
            switch (m.code) {
                case MC_XAB: out += "m xAB\n"; break;
                case MC_XBA: out += "m xBA\n"; break;
                case MC_END: out += "m end\n"; break;
                case MC_FINAL: out += "m final\n"; break;
                case MC_CKPT: out += "m ckpt\n"; break;
                case MC_ROUND: {
                    snprintf(line, sizeof line, "m round mask=%d first=%d flip=%d\n", m.mask, m.arg & ~MOP_FLIP, (m.arg & MOP_FLIP) ? 1 : 0);
                    out += line;
                    int g = ps.gate_begin + (m.arg & ~MOP_FLIP);
                    for (int b = 0; b < 8; ++b) if (m.mask >> b & 1) {
                        const int rc = p.gate_rc[g++];
                        snprintf(line, sizeof line, "g k=%d r=%d c=%d layout=%d\n", (rc >> 13) & 7, (rc >> 6) & 63, rc & 63, (rc >> 12) & 1);
                        out += line;
                    }
                    if (m.arg & MOP_FLIP) {
                        const int rc = p.gate_rc[g++];
                        snprintf(line, sizeof line, "g k=-1 r=%d c=%d layout=%d\n", (rc >> 6) & 63, rc & 63, (rc >> 12) & 1);
                        out += line;
                    }
                    break; }
            }
        }
    }
    return out;
}

}  // namespace ttn
