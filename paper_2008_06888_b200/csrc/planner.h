// planner.h -- host-side pass scheduler for the tropical transfer sweep.
//
// The circuit of Fig. 1(b) has three kinds of operation on the q^L state:
//   g(r,c)   r >= 1 : the single-site max-plus gate (A2) PAPER.md:242 carrying Jv[r-1][c]
//                     (couples row r-1 to row r) on digit c;
//   dh(r,c)         : the field gate (A3) PAPER.md:247, diagonal:  += h[r][c] * sigma_c;
//   dJ(r,c) c < L-1 : the two-site diagonal gate (A4) PAPER.md:251: += Jh[r][c] sigma_c sigma_c+1.
// "The order of operation of these diagonal gates ... can be arbitrary"; gates on
// different digits commute.  Two operations fail to commute only when one is a gate on digit c
// and the other is a gate on c or a diagonal that reads digit c.  Hence the dependency rule
//     g(r,c)  before  dh(r,c), dJ(r,c-1), dJ(r,c)  before  g(r+1,c).
// A pass holds a set of digits in its tile (a contiguous low block [0,lo) that "rides" for
// coalescing plus a high block [a,b)); it may apply, in a legal order, any gate whose digit is
// in the tile and any diagonal (a diagonal only needs the element's own global index).  The
// planner visits a cyclic sequence of overlapping tiles and, in each pass, greedily applies
// every operation that has become legal -- trapezoids/parallelograms over (row, column) as
// deep as the tile allows -- which cuts HBM passes from ceil(L/T) per row to well below one.
//
// Host only; no CUDA.  The same structures are dumped by ttn_plan_describe() and replayed by
// tests/test_planner.py against an independent statement of the rule.
#pragma once
#include <cstdint>
#include <cstdio>
#include <string>
#include <vector>

namespace ttn {

enum OpType : uint8_t { OP_GATE = 0, OP_DH = 1, OP_DJ = 2 };

struct Op {            // 8 bytes, uploaded as-is
    uint8_t type;      // OpType
    uint8_t pos;       // GATE: tile position of the digit (0 .. T-1)
    uint8_t c;         // global column (digit) -- DJ: left digit, pair (c, c+1)
    uint8_t pad;
    uint16_t row;      // lattice row r of the operation
    uint16_t pad2;
};

enum PassFlags : int { PASS_INIT = 1, PASS_REDUCE = 2 };

struct Pass {
    int lo, a, b;          // tile digits = [0,lo) U [a,b), a >= lo; T = lo + (b-a)
    int op_begin, op_end;  // into Plan::ops
    int flags;
    int src_buf, dst_buf;  // -1 = the state V; r >= 0 = checkpoint C_r
    int n_gates;
};

struct Plan {
    int q = 2, L = 0;
    bool row_aligned = false;   // ttn_ground_config: every row boundary is materialised
    std::vector<Pass> passes;
    std::vector<Op> ops;
};

struct TileSpec { int lo, a, b; };

class Scheduler {
  public:
    Scheduler(int L, bool has_field) : L_(L), has_field_(has_field), grow_(L, 1),
        dh_(L * L, 0), dj_(L * (L > 1 ? L - 1 : 1), 0) {
        if (!has_field_) for (auto& x : dh_) x = 1;   // nothing to apply
    }
    bool done() const {
        for (int c = 0; c < L_; ++c) if (grow_[c] != L_) return false;
        for (auto x : dh_) if (!x) return false;
        for (int r = 0; r < L_; ++r) for (int c = 0; c + 1 < L_; ++c) if (!dj_[r * (L_ - 1) + c]) return false;
        return true;
    }
    bool row_done(int r) const {   // all of row r's gates and diagonals applied
        for (int c = 0; c < L_; ++c) if (grow_[c] < r + 1 || !dh_[r * L_ + c]) return false;
        for (int c = 0; c + 1 < L_; ++c) if (!dj_[r * (L_ - 1) + c]) return false;
        return true;
    }
    // Greedily apply everything legal for tile digits [0,lo) U [a,b) with rows <= max_row.
    // Appends to ops; returns number of gates applied.
    int run_pass(const TileSpec& t, int max_row, std::vector<Op>& ops) {
        int gates = 0;
        bool progress = true;
        auto in_tile = [&](int c) { return c < t.lo || (c >= t.a && c < t.b); };
        auto pos_of = [&](int c) { return c < t.lo ? c : t.lo + (c - t.a); };
        while (progress) {
            progress = false;
            for (int c = 0; c < L_; ++c) {
                if (!in_tile(c)) continue;
                int r = grow_[c] - 1;                       // row currently complete on digit c
                if (r > max_row) continue;
                if (!dh_[r * L_ + c]) { dh_[r * L_ + c] = 1; ops.push_back({OP_DH, 0, (uint8_t)c, 0, (uint16_t)r, 0}); progress = true; }
                for (int cc = c - 1; cc <= c; ++cc) {
                    if (cc < 0 || cc + 1 >= L_) continue;
                    if (grow_[cc] == grow_[cc + 1] && grow_[cc] - 1 == r && !dj_[r * (L_ - 1) + cc]) {
                        dj_[r * (L_ - 1) + cc] = 1;
                        ops.push_back({OP_DJ, 0, (uint8_t)cc, 0, (uint16_t)r, 0});
                        progress = true;
                    }
                }
            }
            for (int c = 0; c < L_; ++c) {
                if (!in_tile(c)) continue;
                int r = grow_[c];                           // next gate row on digit c
                if (r >= L_ || r > max_row) continue;
                bool ok = dh_[(r - 1) * L_ + c] != 0;
                if (c > 0) ok = ok && dj_[(r - 1) * (L_ - 1) + c - 1];
                if (c + 1 < L_) ok = ok && dj_[(r - 1) * (L_ - 1) + c];
                if (!ok) continue;
                grow_[c] += 1;
                ops.push_back({OP_GATE, (uint8_t)pos_of(c), (uint8_t)c, 0, (uint16_t)r, 0});
                ++gates; progress = true;
            }
        }
        return gates;
    }
  private:
    int L_; bool has_field_;
    std::vector<int> grow_;            // grow[c] = rows complete on digit c (row 0 needs no gate)
    std::vector<uint8_t> dh_, dj_;
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
inline Plan make_plan(int q, int L, bool has_field, bool row_aligned, int Tmax, int ride) {
    Plan best;
    int wh = Tmax - ride;
    int s_lo = 1, s_hi = wh;
    if (Tmax >= L) { s_lo = s_hi = 1; }
    if (row_aligned) { s_lo = s_hi = wh; }
    bool have = false;
    for (int stride = s_lo; stride <= s_hi; ++stride) {
        std::vector<TileSpec> cyc = tile_cycle(L, Tmax, ride, stride);
        Plan p; p.q = q; p.L = L; p.row_aligned = row_aligned;
        Scheduler s(L, has_field);
        size_t k = 0; int row = 0; bool first = true; int idle = 0;
        int cur_src = -1;
        while (first || !s.done()) {   // the INIT pass exists even when there is nothing to apply
            const TileSpec& t = cyc[k % cyc.size()]; ++k;
            Pass ps{t.lo, t.a, t.b, (int)p.ops.size(), 0, 0, -1, -1, 0};
            ps.n_gates = s.run_pass(t, row_aligned ? row : L, p.ops);
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

inline std::string describe(const Plan& p) {
    std::string out;
    char line[160];
    snprintf(line, sizeof line, "plan q=%d L=%d row_aligned=%d passes=%zu ops=%zu\n", p.q, p.L,
             (int)p.row_aligned, p.passes.size(), p.ops.size());
    out += line;
    for (size_t i = 0; i < p.passes.size(); ++i) {
        const Pass& ps = p.passes[i];
        snprintf(line, sizeof line, "pass %zu lo=%d a=%d b=%d flags=%d src=%d dst=%d gates=%d nops=%d\n",
                 i, ps.lo, ps.a, ps.b, ps.flags, ps.src_buf, ps.dst_buf, ps.n_gates, ps.op_end - ps.op_begin);
        out += line;
        for (int k = ps.op_begin; k < ps.op_end; ++k) {
            const Op& o = p.ops[k];
            snprintf(line, sizeof line, "op %s r=%d c=%d pos=%d\n",
                     o.type == OP_GATE ? "g" : (o.type == OP_DH ? "dh" : "dJ"), o.row, o.c, o.pos);
            out += line;
        }
    }
    return out;
}

}  // namespace ttn
