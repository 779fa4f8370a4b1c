// host_model.hpp — host-side preparation of one diagram (not on the timed path).
// Product code (libmcqed.so); written from PAPER.md and DESIGN.md, shares nothing with oracle/.
//
//   VertexGraph   : the graph, its validity (1PI), class (k,m,n) [PAPER.md:104], canonical index
//   Segment       : a UV-divergent subgraph as a position segment [PAPER.md:53,:59]
//   ForestTerms   : forests and the terms of the forest-like formula [PAPER.md:63; O1]
//   Piece         : a forest element with its maximal children shrunk [DESIGN.md R5, O2, O3]
//   SamplerTables : Deg(s), invDeg(s), Z(s), C of Eq.(1) [PAPER.md:74-78; S2, S5]
#pragma once
#include <algorithm>
#include <array>
#include <cstdint>
#include <cstring>
#include <map>
#include <mutex>
#include <vector>

#include "device_layout.h"

namespace mq {

struct VertexGraph {
  int L = 0, e = 0, M = 0, npos = 0;
  int ca[MQ_MAXL], cb[MQ_MAXL];  // chords, sorted by first end
  int mate[2 * MQ_MAXL + 1];     // partner position (-1 at e)
  int chordOf[2 * MQ_MAXL + 1];  // chord index at a position (-1 at e)

  // returns false if (loops, ext, chords) is not a valid 1PI vertex graph
  bool build(int loops, int ext, const int32_t *a, const int32_t *b) {
    if (loops < 1 || loops > MQ_MAXL) return false;
    L = loops; e = ext; M = 3 * L; npos = 2 * L + 1;
    if (e < 0 || e >= npos) return false;
    std::vector<std::pair<int, int>> ch;
    for (int i = 0; i < L; i++) {
      int x = std::min(a[i], b[i]), y = std::max(a[i], b[i]);
      if (x < 0 || y >= npos || x == y || x == e || y == e) return false;
      ch.emplace_back(x, y);
    }
    std::sort(ch.begin(), ch.end());
    std::fill(mate, mate + npos, -1); std::fill(chordOf, chordOf + npos, -1);
    for (int i = 0; i < L; i++) {
      ca[i] = ch[i].first; cb[i] = ch[i].second;
      if (chordOf[ca[i]] >= 0 || chordOf[cb[i]] >= 0) return false;
      chordOf[ca[i]] = chordOf[cb[i]] = i; mate[ca[i]] = cb[i]; mate[cb[i]] = ca[i];
    }
    for (int t = 0; t < 2 * L; t++) if (!lineCovered(t, 0, 2 * L)) return false;
    return true;
  }
  // electron line t spanned by a chord lying inside [lo,hi]
  bool lineCovered(int t, int lo, int hi) const {
    for (int i = 0; i < L; i++) if (ca[i] >= lo && cb[i] <= hi && ca[i] <= t && t < cb[i]) return true;
    return false;
  }
  void classKMN(int &k, int &m, int &n) const {
    int across = 0, left = 0, right = 0;
    for (int i = 0; i < L; i++) { if (cb[i] < e) left++; else if (ca[i] > e) right++; else across++; }
    k = across; m = std::max(left, right); n = std::min(left, right);
  }
  std::array<int8_t, 12> key() const {
    std::array<int8_t, 12> k{}; k[0] = (int8_t)e;
    for (int i = 0; i < L; i++) { k[1 + 2 * i] = (int8_t)ca[i]; k[2 + 2 * i] = (int8_t)cb[i]; }
    return k;
  }
  // position in the canonical list of valid graphs of this loop order (ascending e, lexicographic chords)
  int canonicalId() const;
};

namespace detail {
inline void matchings(int L, int e, std::vector<int> &free_pos, std::array<int8_t, 12> &cur, int depth, std::vector<std::array<int8_t, 12>> &out) {
  if (free_pos.empty()) {
    int32_t a[MQ_MAXL], b[MQ_MAXL];
    for (int i = 0; i < L; i++) { a[i] = cur[1 + 2 * i]; b[i] = cur[2 + 2 * i]; }
    VertexGraph g;
    if (g.build(L, e, a, b)) out.push_back(cur);
    return;
  }
  int first = free_pos.front();
  for (size_t j = 1; j < free_pos.size(); j++) {
    int second = free_pos[j];
    std::vector<int> rest;
    for (size_t q = 1; q < free_pos.size(); q++) if (q != j) rest.push_back(free_pos[q]);
    cur[1 + 2 * depth] = (int8_t)first; cur[2 + 2 * depth] = (int8_t)second;
    matchings(L, e, rest, cur, depth + 1, out);
  }
}
inline const std::vector<std::array<int8_t, 12>> &canonicalList(int L) {
  static std::mutex mtx; static std::map<int, std::vector<std::array<int8_t, 12>>> cache;
  std::lock_guard<std::mutex> lock(mtx);
  auto it = cache.find(L);
  if (it != cache.end()) return it->second;
  std::vector<std::array<int8_t, 12>> all;
  for (int e = 0; e <= 2 * L; e++) {
    std::vector<int> fp;
    for (int p = 0; p <= 2 * L; p++) if (p != e) fp.push_back(p);
    std::array<int8_t, 12> cur{}; cur[0] = (int8_t)e;
    matchings(L, e, fp, cur, 0, all);
  }
  return cache[L] = std::move(all);
}
}  // namespace detail

inline int VertexGraph::canonicalId() const {
  const auto &lst = detail::canonicalList(L);
  auto k = key();
  for (size_t i = 0; i < lst.size(); i++) if (lst[i] == k) return (int)i;
  return -1;
}

struct Segment {
  int lo, hi; bool vertexLike;
  bool has(int pos) const { return lo <= pos && pos <= hi; }
  bool within(const Segment &o) const { return o.lo <= lo && hi <= o.hi; }
  bool operator==(const Segment &o) const { return lo == o.lo && hi == o.hi; }
};

struct ForestTerms {
  std::vector<Segment> subs;        // ascending (lo,hi)
  std::vector<uint32_t> forests;    // ascending bitmask, empty forest included
  struct Term { uint32_t forest; int gprime; int sign; };
  std::vector<Term> terms;

  void enumerate(const VertexGraph &g) {
    subs.clear(); forests.clear(); terms.clear();
    for (int lo = 0; lo <= 2 * g.L; lo++) for (int hi = lo + 1; hi <= 2 * g.L; hi++) {
      if (lo == 0 && hi == 2 * g.L) continue;
      int external = 0;
      for (int x = lo; x <= hi; x++) external += (x == g.e) || (x != g.e && (g.mate[x] < lo || g.mate[x] > hi));
      if (external > 1) continue;
      bool opi = true;
      for (int t = lo; t < hi && opi; t++) opi = g.lineCovered(t, lo, hi);
      if (opi) subs.push_back({lo, hi, external == 1});
    }
    int n = (int)subs.size();
    for (uint32_t m = 0; m < (1u << n); m++) {
      bool ok = true;
      for (int i = 0; i < n && ok; i++) if (m >> i & 1) for (int j = i + 1; j < n && ok; j++) if (m >> j & 1) {
        const Segment &x = subs[i], &y = subs[j];
        ok = x.within(y) || y.within(x) || x.hi < y.lo || y.hi < x.lo;
      }
      if (ok) forests.push_back(m);
    }
    for (uint32_t f : forests) {
      int sign = (__builtin_popcount(f) & 1) ? -1 : 1;   // (-1)^{|F|-1}, |F| counts G
      terms.push_back({f, -1, sign});
      for (int i = 0; i < n; i++) if ((f >> i & 1) && subs[i].vertexLike && subs[i].has(g.e)) terms.push_back({f, i, sign});
    }
  }
  // maximal members of forest f strictly inside seg (indices into subs, ascending lo)
  std::vector<int> childrenOf(uint32_t f, const Segment &seg) const {
    std::vector<int> inside, out;
    for (int i = 0; i < (int)subs.size(); i++) if ((f >> i & 1) && subs[i].within(seg) && !(subs[i] == seg)) inside.push_back(i);
    for (int i : inside) {
      bool maximal = true;
      for (int j : inside) if (j != i && subs[i].within(subs[j])) maximal = false;
      if (maximal) out.push_back(i);
    }
    return out;
  }
};

// ---------------------------------------------------------------------------------------------
struct Piece {
  enum ElemKind { VERT_CHORD, VERT_FREE, SLOT };
  struct Elem { ElemKind kind; int chord; int slot; };      // chord: local own-chord index
  struct Slot { bool insertion; int line; int child; uint32_t eps; int sgn; };
  Segment seg{};
  std::vector<Segment> kids;
  std::vector<int> ownChord;     // global chord indices
  std::vector<Slot> slots;
  std::vector<Elem> elems;       // path order
  int nS = 0;
  std::vector<int> patbit;       // per child: bit in the compressed pattern (S-children), -1 for V

  int kidAt(int pos) const { for (int c = 0; c < (int)kids.size(); c++) if (kids[c].has(pos)) return c; return -1; }

  void build(const VertexGraph &g, const Segment &s, const std::vector<Segment> &children) {
    seg = s; kids = children; ownChord.clear(); slots.clear(); elems.clear(); patbit.clear(); nS = 0;
    for (auto &k : kids) patbit.push_back(k.vertexLike ? -1 : nS++);
    std::vector<int> local(g.L, -1);
    for (int i = 0; i < g.L; i++) {
      if (!(seg.has(g.ca[i]) && seg.has(g.cb[i]))) continue;
      int ka = kidAt(g.ca[i]), kb = kidAt(g.cb[i]);
      if (ka >= 0 && ka == kb) continue;
      local[i] = (int)ownChord.size(); ownChord.push_back(i);
    }
    int freePos = -1;
    if (seg.vertexLike) {
      if (seg.has(g.e)) freePos = g.e;
      else for (int x = seg.lo; x <= seg.hi; x++) if (!seg.has(g.mate[x])) freePos = x;
    }
    auto chordLeaving = [&](const Segment &k) {
      for (int x = k.lo; x <= k.hi; x++) if (x != g.e && !k.has(g.mate[x])) return g.chordOf[x];
      return -1;
    };
    for (int pos = seg.lo; pos <= seg.hi;) {
      int k = kidAt(pos);
      if (k >= 0 && !kids[k].vertexLike) {
        slots.push_back({true, kids[k].lo - 1, k, 0u, 0});
        elems.push_back({SLOT, -1, (int)slots.size() - 1});
        pos = kids[k].hi + 1;
      } else if (k >= 0) {
        if (freePos >= 0 && kids[k].has(freePos)) elems.push_back({VERT_FREE, -1, -1});
        else elems.push_back({VERT_CHORD, local[chordLeaving(kids[k])], -1});
        pos = kids[k].hi + 1;
      } else {
        if (pos == freePos) elems.push_back({VERT_FREE, -1, -1});
        else elems.push_back({VERT_CHORD, local[g.chordOf[pos]], -1});
        pos++;
      }
      if (pos <= seg.hi) {
        slots.push_back({false, pos - 1, -1, 0u, 0});
        elems.push_back({SLOT, -1, (int)slots.size() - 1});
      }
    }
    for (auto &sl : slots) {
      for (int j = 0; j < (int)ownChord.size(); j++) { int i = ownChord[j]; if (g.ca[i] <= sl.line && sl.line < g.cb[i]) sl.eps |= 1u << j; }
      sl.sgn = sl.line < g.e ? -1 : 1;
    }
  }
  // bit mask (over the M line indices) of the lines owned by this piece
  uint32_t lineMask(const VertexGraph &g) const {
    uint32_t m = 0;
    for (auto &sl : slots) if (!sl.insertion) m |= 1u << sl.line;
    for (int i : ownChord) m |= 1u << (2 * g.L + i);
    return m;
  }
  // cycle rank of the line subset s (restricted to own lines) in the piece graph (children shrunk to points)
  int loopsOf(const VertexGraph &g, uint32_t s) const {
    int root[32];
    for (int i = 0; i < 32; i++) root[i] = i;
    auto node = [&](int pos) { int k = kidAt(pos); return k >= 0 ? 16 + k : pos; };
    auto find = [&](int x) { while (root[x] != x) x = root[x] = root[root[x]]; return x; };
    uint32_t touched = 0; int edges = 0, merges = 0;
    auto add = [&](int u, int v) { edges++; touched |= 1u << u | 1u << v; int a = find(u), b = find(v); if (a != b) { root[a] = b; merges++; } };
    for (auto &sl : slots) if (!sl.insertion && (s >> sl.line & 1)) add(node(sl.line), node(sl.line + 1));
    for (int i : ownChord) if (s >> (2 * g.L + i) & 1) add(node(g.ca[i]), node(g.cb[i]));
    int verts = __builtin_popcount(touched);
    return edges - verts + (verts - merges);   // E - V + C, C = V - merges
  }
};

// ---------------------------------------------------------------------------------------------
struct SamplerTables {
  int M = 0;
  std::vector<double> deg, invdeg, Z;
  double C = 0;

  // dfloor_ir: the value on sets whose I-closure is the whole graph (the soft-photon sets of PAPER.md:78); <= 0: same as dfloor
  void build(const VertexGraph &g, const ForestTerms &ft, double dfloor, double dcap, double dfloor_ir_in = 0.0) {
    const double dfloor_ir = dfloor_ir_in > 0.0 ? dfloor_ir_in : dfloor;
    M = g.M; size_t n = (size_t)1 << M; uint32_t full = (uint32_t)n - 1;
    deg.assign(n, 0.0); invdeg.assign(n, 0.0); Z.assign(n, 0.0);
    // pieces of the maximal forests only: shrinking more never lowers the loop count (S5)
    std::vector<std::vector<Piece>> sets;
    Segment whole{0, 2 * g.L, true};
    for (uint32_t f : ft.forests) {
      bool maximal = true;
      for (uint32_t h : ft.forests) if (h != f && (h & f) == f) maximal = false;
      if (!maximal) continue;
      std::vector<Piece> ps;
      auto mk = [&](const Segment &s) { std::vector<Segment> kids; for (int k : ft.childrenOf(f, s)) kids.push_back(ft.subs[k]); Piece p; p.build(g, s, kids); ps.push_back(p); };
      mk(whole);
      for (int i = 0; i < (int)ft.subs.size(); i++) if (f >> i & 1) mk(ft.subs[i]);
      sets.push_back(std::move(ps));
    }
    // per piece: loop count of every subset of its own lines (memoised)
    struct Memo { uint32_t mask; std::vector<int> bits; std::vector<int8_t> loops; };
    std::vector<std::vector<Memo>> memo(sets.size());
    for (size_t f = 0; f < sets.size(); f++) for (auto &p : sets[f]) {
      Memo m; m.mask = p.lineMask(g);
      for (int b = 0; b < M; b++) if (m.mask >> b & 1) m.bits.push_back(b);
      size_t cnt = (size_t)1 << m.bits.size(); m.loops.resize(cnt);
      for (size_t sub = 0; sub < cnt; sub++) {
        uint32_t s = 0;
        for (size_t j = 0; j < m.bits.size(); j++) if (sub >> j & 1) s |= 1u << m.bits[j];
        m.loops[sub] = (int8_t)p.loopsOf(g, s);
      }
      memo[f].push_back(std::move(m));
    }
    uint32_t emask = (1u << (2 * g.L)) - 1;
    std::vector<uint32_t> path(g.L);
    for (int i = 0; i < g.L; i++) { uint32_t m = 0; for (int t = g.ca[i]; t < g.cb[i]; t++) m |= 1u << t; path[i] = m; }
    for (uint32_t s = 1; s < full; s++) {
      uint32_t sb = s;   // I-closure
      for (int i = 0; i < g.L; i++) if ((s & path[i]) == path[i]) sb |= 1u << (2 * g.L + i);
      double d;
      if (sb == full) d = dfloor_ir;
      else {
        int best = 0;
        for (size_t f = 0; f < sets.size(); f++) {
          int tot = 0;
          for (auto &m : memo[f]) {
            size_t sub = 0;
            for (size_t j = 0; j < m.bits.size(); j++) if (sb >> m.bits[j] & 1) sub |= (size_t)1 << j;
            tot += m.loops[sub];
          }
          best = std::max(best, tot);
        }
        d = (double)__builtin_popcount(sb) - 0.5 * (double)__builtin_popcount(sb & emask) - 2.0 * (double)best;
        d = std::min(std::max(d, dfloor), dcap);
      }
      deg[s] = d; invdeg[s] = 1.0 / d;
    }
    // Z(0)=1; Z(s) = invDeg(s) * sum_{x in s, ascending} Z(s \ x)   (S2: order is part of the spec)
    Z[0] = 1.0;
    for (uint32_t s = 1; s < full; s++) {
      double acc = 0.0;
      for (int x = 0; x < M; x++) if (s >> x & 1) acc = acc + Z[s & ~(1u << x)];
      Z[s] = acc * invdeg[s];
    }
    double tot = 0.0;
    for (int x = 0; x < M; x++) tot = tot + Z[full & ~(1u << x)];
    Z[full] = tot; C = 1.0 / tot;
  }
};

}  // namespace mq
