// coef_gen.hpp — numerator tables of one piece under one operator (host, prepare time).
// Product code (libmcqed.so); shares nothing with oracle/.
//
// DESIGN.md O3-O5. In the rest frame p=(m,0,0,0), m=1, Dirac representation, every factor of the
// gamma string of a piece is a generalised permutation matrix (one non-zero entry i^k per column)
// or a block projector:
//     line t, unpaired :  (A_t pslash + m) = g_t (P+ + r_t P-),   g_t = 2-x_t, r_t = x_t/g_t, x_t = 1-A_t
//     kappaslash, vertices, free vertex, q-slot : gamma^rho
// So for fixed Lorentz indices a basis spinor follows ONE path through the string, picking up a
// phase, and the block (upper/lower) it is in at an unpaired line decides P+ or P-. The coefficient
// of a monomial is the signed count of such paths: exact integer arithmetic, no matrix products.
//
// Output format ("families"): for a fixed role of every slot
// {binary line, insertion a-part, insertion b*p-part, Wick-paired, q-slot} and a fixed P+/P- choice
// of the outer binary lines, ALL pairings of the paired slots times ALL 2^kd choices of the inner
// binary lines, as one dense coefficient block the kernel evaluates with static register indexing.
#pragma once
#include <atomic>
#include <chrono>
#include <cstdio>
#include <complex>
#include <cstdlib>
#include <cstring>
#include <functional>
#include <thread>

#include "host_model.hpp"

namespace mq {

struct Family {
  int c = 0, kd = 0, pattern = 0, out = 0;
  std::vector<uint8_t> paired, inner;
  std::vector<uint8_t> scal;       // kind<<4 | slot
  std::vector<double> coef;        // stream order (see device_layout.h), incl. the closing (sum |c|, -) unit of every kd >= 3 block
  int64_t nonzero = 0, n_coef = 0; // non-zero / stored numerator coefficients (closing units not counted)
};
struct TableBuild { int nout = 1; std::vector<Family> fams; int64_t n_stored = 0, n_nonzero = 0; };

namespace detail {
// column action of gamma^rho on basis spinor s: gamma^rho e_s = i^PH e_DST   (Dirac representation)
static const int8_t G_DST[4][4] = {{0, 1, 2, 3}, {3, 2, 1, 0}, {3, 2, 1, 0}, {2, 3, 0, 1}};
static const int8_t G_PH[4][4] = {{0, 0, 2, 2}, {2, 2, 0, 0}, {3, 1, 1, 3}, {2, 0, 0, 2}};

enum { W_FIX = MQ_W_FIX, W_OPEN = MQ_W_OPEN, W_CLOSE = MQ_W_CLOSE, W_BIN = MQ_W_BIN, W_G0 = MQ_W_G0 };
using WElem = MqWElem;
using CountUnit = MqCountUnit;

struct Variant {               // one trace of the operator functional
  int freeIdx, qIdx, prepend, append;     // Lorentz index of the free vertex / q-slot; extra gamma applied first / last (-1 none)
  std::complex<double> w[4];              // weight per start spinor (0 = not used)
  int out;
};

// integer path counting on the host (the same walk runs as a CUDA kernel in prep_kernel.cu)
struct Walker {
  const WElem *el; int n; int start;
  int8_t rho[16];
  int32_t *acc;   // [2^k][2]
  void go(int pos, int s, int ph, uint32_t sig) {
    for (; pos < n; pos++) {
      const WElem e = el[pos];
      switch (e.type) {
        case W_FIX: ph += G_PH[e.arg][s]; s = G_DST[e.arg][s]; break;
        case W_G0: ph += (s >= 2) ? 2 : 0; break;
        case W_BIN: sig |= (uint32_t)(s >= 2) << e.arg; break;
        case W_CLOSE: { int r = rho[e.arg]; ph += G_PH[r][s] + (r ? 2 : 0); s = G_DST[r][s]; break; }
        case W_OPEN:
          for (int r = 0; r < 4; r++) { rho[e.arg] = (int8_t)r; go(pos + 1, G_DST[r][s], ph + G_PH[r][s], sig); }
          return;
      }
    }
    if (s != start) return;
    acc[2 * sig + (ph & 1)] += (ph & 2) ? -1 : 1;
  }
};

inline std::vector<Variant> variantsFor(int op, bool sType, bool hasQ) {
  using cd = std::complex<double>;
  std::vector<Variant> v;
  const cd i(0, 1);
  auto L = [&](double sc) { v.push_back({0, -1, -1, -1, {cd(0.5 * sc), cd(0.5 * sc), 0, 0}, 0}); };
  // U_V = -(1/12) sum_j Tr[gamma^j X^j] is a multiple of 1/12: tables of U and (L-U) on vertex-like pieces store
  // 12*coefficient (exactly representable); the kernel divides by 12 once in its working precision
  auto U = [&](double sc) { for (int j = 1; j <= 3; j++) v.push_back({j, -1, -1, j, {cd(-sc), cd(-sc), cd(-sc), cd(-sc)}, 0}); };
  if (sType) {            // U on an electron self-energy: a = Tr S/4, b = Tr[gamma^0 S]/4
    v.push_back({-1, -1, -1, -1, {0.25, 0.25, 0.25, 0.25}, 0});
    v.push_back({-1, -1, -1, 0, {0.25, 0.25, 0.25, 0.25}, 1});
    return v;
  }
  switch (op) {
    case MQ_OP_L: L(1); break;
    case MQ_OP_U: U(1); break;
    case MQ_OP_LMU: L(12); U(-1); break;      // 12 (L - U)
    case MQ_OP_A:
      if (!hasQ) {        // [ (g2 X1 - X1 g2)_00 - (..)_11 ]/(4i) - (X0_00 + X0_11)/2      (O4)
        v.push_back({1, -1, -1, 2, {-0.25 * i, 0.25 * i, 0, 0}, 0});
        v.push_back({1, -1, 2, -1, {0.25 * i, -0.25 * i, 0, 0}, 0});
        v.push_back({0, -1, -1, -1, {-0.5, -0.5, 0, 0}, 0});
      } else {            // -i [ Y12_00 - Y12_11 ]
        v.push_back({1, 2, -1, -1, {-i, i, 0, 0}, 0});
      }
      break;
  }
  return v;
}

// all perfect matchings of {0..2c-1} in canonical order: the first free element pairs with every later one
inline void allPairings(int n2, std::vector<std::vector<std::pair<int, int>>> &out) {
  std::vector<std::pair<int, int>> cur;
  std::vector<int> used(n2, 0);
  std::function<void()> rec = [&]() {
    int f = 0; while (f < n2 && used[f]) f++;
    if (f == n2) { out.push_back(cur); return; }
    used[f] = 1;
    for (int s = f + 1; s < n2; s++) if (!used[s]) { used[s] = 1; cur.emplace_back(f, s); rec(); cur.pop_back(); used[s] = 0; }
    used[f] = 0;
  };
  rec();
}
}  // namespace detail

enum Role : uint8_t { R_BIN, R_INS_A, R_INS_BP, R_PAIRED, R_Q };

struct RoleJob { std::vector<uint8_t> role; int c; bool hasQ; };

// optional accelerator: counts all units on the GPU (prep_kernel.cu); returns 0 on success
using GpuCountFn = int (*)(const detail::CountUnit *units, size_t nunits, int32_t *counts, size_t nints);

// maxGrade: own grades above it can never reach the integrand (only total grades c < L enter O6)
inline TableBuild buildTable(const Piece &p, int op, int nthreads, int maxGrade, GpuCountFn gpuCount = nullptr) {
  using namespace detail;
  TableBuild tb;
  const bool sType = !p.seg.vertexLike;
  tb.nout = sType ? 2 : 1;
  const int nslot = (int)p.slots.size(), nch = (int)p.ownChord.size();
  int maxc = std::min(nslot / 2, maxGrade);
  if ((op == MQ_OP_A || op == MQ_OP_LMU) && p.nS == 0) maxc = std::min(maxc, nch - 1);  // top grade ~ gamma^mu: killed (O4)
  // ---- enumerate slot roles ----
  std::vector<RoleJob> jobs;
  {
    std::vector<uint8_t> role(nslot);
    std::function<void(int, int, bool)> rec = [&](int s, int npaired, bool usedQ) {
      if (s == nslot) { if (npaired % 2 == 0 && npaired / 2 <= maxc) jobs.push_back({role, npaired / 2, usedQ}); return; }
      if (!p.slots[s].insertion) { role[s] = R_BIN; rec(s + 1, npaired, usedQ); }
      else { role[s] = R_INS_A; rec(s + 1, npaired, usedQ); role[s] = R_INS_BP; rec(s + 1, npaired, usedQ); }
      if (npaired + 1 <= 2 * maxc) { role[s] = R_PAIRED; rec(s + 1, npaired + 1, usedQ); }
      if (op == MQ_OP_A && !usedQ) { role[s] = R_Q; rec(s + 1, npaired, true); }
    };
    rec(0, 0, false);
  }
  std::vector<std::vector<std::vector<std::pair<int, int>>>> pairingsOf(maxc + 1);
  for (int c = 0; c <= maxc; c++) allPairings(2 * c, pairingsOf[c]);

  const bool timing = std::getenv("MCQED_PREPARE_TIMING") != nullptr;
  auto tick = std::chrono::steady_clock::now();
  auto lap = [&](const char *what) { if (timing) { auto now = std::chrono::steady_clock::now(); std::fprintf(stderr, "[mcqed prepare] %s %.1f ms\n", what, std::chrono::duration<double, std::milli>(now - tick).count()); tick = now; } };
  // ---- phase A: one counting unit per (job, pairing, variant, start spinor) ----
  struct UnitMeta { uint32_t job, pairing; int out; std::complex<double> w; };
  struct JobInfo { std::vector<int> binSlots, pairedSlots, atSlots; int qSlot = -1, pattern = 0; size_t firstUnit = 0, nUnits = 0; };
  std::vector<CountUnit> units; std::vector<UnitMeta> meta; std::vector<JobInfo> info(jobs.size());
  uint64_t nints = 0;
  for (size_t j = 0; j < jobs.size(); j++) {
    const RoleJob &job = jobs[j]; JobInfo &ji = info[j];
    for (int s = 0; s < nslot; s++) {
      Role r = (Role)job.role[s];
      if (r == R_BIN) ji.binSlots.push_back(s);
      if (r == R_PAIRED) ji.pairedSlots.push_back(s);
      if (r == R_INS_BP) ji.atSlots.push_back(s);
      if (r == R_Q) ji.qSlot = s;
      if (p.slots[s].insertion && r != R_INS_A) ji.pattern |= 1 << p.patbit[p.slots[s].child];
    }
    const int k = (int)ji.binSlots.size(), c = job.c;
    const auto &pairings = pairingsOf[c];
    const auto variants = variantsFor(op, sType, job.hasQ);
    std::vector<int> pairIdOfSlot(nslot, -1), binIdx(nslot, -1);
    for (int b = 0; b < k; b++) binIdx[ji.binSlots[b]] = b;
    ji.firstUnit = units.size();
    for (size_t pi = 0; pi < pairings.size(); pi++) {
      std::vector<int> firstOfPair(nslot, 0);
      for (int q = 0; q < c; q++) {
        pairIdOfSlot[ji.pairedSlots[pairings[pi][q].first]] = nch + q; firstOfPair[ji.pairedSlots[pairings[pi][q].first]] = 1;
        pairIdOfSlot[ji.pairedSlots[pairings[pi][q].second]] = nch + q;
      }
      for (const Variant &var : variants) {
        CountUnit u; std::memset(&u, 0, sizeof u);
        int n = 0;
        auto push = [&](int type, int arg) { u.el[n].type = (uint8_t)type; u.el[n].arg = (uint8_t)arg; n++; };
        if (var.prepend >= 0) push(W_FIX, var.prepend);
        std::vector<int> chordSeen(nch, 0);
        for (const auto &e : p.elems) {
          if (e.kind == Piece::VERT_FREE) push(W_FIX, var.freeIdx);
          else if (e.kind == Piece::VERT_CHORD) { push(chordSeen[e.chord] ? W_CLOSE : W_OPEN, e.chord); chordSeen[e.chord] = 1; }
          else {
            int s = e.slot;
            switch ((Role)job.role[s]) {
              case R_BIN: push(W_BIN, binIdx[s]); break;
              case R_INS_A: break;
              case R_INS_BP: push(W_G0, 0); break;
              case R_PAIRED: push(firstOfPair[s] ? W_OPEN : W_CLOSE, pairIdOfSlot[s]); break;
              case R_Q: push(W_FIX, var.qIdx); break;
            }
          }
        }
        if (var.append >= 0) push(W_FIX, var.append);
        u.n = (uint8_t)n; u.npairs = (uint8_t)(nch + c); u.nsig = 1u << k;
        for (int a = 0; a < 4; a++) {
          if (var.w[a] == std::complex<double>(0, 0)) continue;
          u.start = (uint8_t)a; u.off = nints; nints += 2ull * u.nsig;
          units.push_back(u); meta.push_back({(uint32_t)j, (uint32_t)pi, var.out, var.w[a]});
        }
      }
    }
    ji.nUnits = units.size() - ji.firstUnit;
  }
  lap("units");
  // ---- phase B: count paths (GPU if offered, else host threads) ----
  std::vector<int32_t> counts(nints, 0);
  bool counted = false;
  if (gpuCount && !units.empty()) counted = gpuCount(units.data(), units.size(), counts.data(), counts.size()) == 0;
  auto parallelFor = [&](size_t n, const std::function<void(size_t)> &fn) {
    std::atomic<size_t> next{0};
    auto worker = [&]() { for (;;) { size_t i = next.fetch_add(1); if (i >= n) break; fn(i); } };
    int nt = std::max(1, std::min<int>(nthreads, (int)n));
    std::vector<std::thread> pool;
    for (int t = 1; t < nt; t++) pool.emplace_back(worker);
    worker();
    for (auto &t : pool) t.join();
  };
  if (!counted) {
    std::fill(counts.begin(), counts.end(), 0);
    parallelFor(units.size(), [&](size_t i) {
      Walker w; w.el = units[i].el; w.n = units[i].n; w.start = units[i].start; w.acc = counts.data() + units[i].off;
      w.go(0, units[i].start, 0, 0u);
    });
  }
  lap(counted ? "count(gpu)" : "count(host)");
  // ---- phase C: coefficients and families, job by job ----
  std::vector<std::vector<Family>> famsOf(jobs.size());
  parallelFor(jobs.size(), [&](size_t j) {
    const JobInfo &ji = info[j];
    const int k = (int)ji.binSlots.size(), c = jobs[j].c;
    const size_t npair = pairingsOf[c].size(), nsig = (size_t)1 << k;
    std::vector<double> cm((size_t)tb.nout * npair * nsig, 0.0);   // [out][pairing][sigma]
    double pref = 1.0;
    for (int i = 0; i < nch; i++) pref *= -0.25;
    for (int i = 0; i < c; i++) pref *= -0.5;
    for (size_t ui = ji.firstUnit; ui < ji.firstUnit + ji.nUnits; ui++) {
      const UnitMeta &m = meta[ui];
      const int32_t *cnt = counts.data() + units[ui].off;
      double *dst = &cm[((size_t)m.out * npair + m.pairing) * nsig];
      // Re[w (re + i im)]: weights are dyadic and counts are integers, so every term is exact
      for (size_t sg = 0; sg < nsig; sg++) dst[sg] += pref * (m.w.real() * (double)cnt[2 * sg] - m.w.imag() * (double)cnt[2 * sg + 1]);
    }
    int kdcap = mq_kd_max(c);
    if (const char *env = std::getenv("MCQED_KD_CAP")) kdcap = std::min(kdcap, std::max(0, atoi(env)));   // experiments only
    const int kd = std::min(k, kdcap), ko = k - kd;
    const size_t ninner = (size_t)1 << kd, half = ninner >> 1;
    for (int out = 0; out < tb.nout; out++)
      for (size_t so = 0; so < ((size_t)1 << ko); so++) {
        Family f; f.c = c; f.kd = kd; f.pattern = ji.pattern; f.out = out;
        bool any = false;
        for (size_t pi = 0; pi < npair; pi++) {
          const double *src = &cm[((size_t)out * npair + pi) * nsig];
          auto at = [&](size_t si) { return src[so | (si << ko)]; };   // outer bits low, inner bits high
          if (kd == 0) { f.coef.push_back(at(0)); f.n_coef++; if (at(0) != 0.0) f.nonzero++; continue; }
          if (kd <= 4) for (size_t jj = 0; jj < half; jj++) { f.coef.push_back(at(jj)); f.coef.push_back(at(jj + half)); }
          else for (size_t top = 0; top < (ninner >> 4); top++)          // kd = 5, 6: sub-blocks of kd = 4, top bits ascending
            for (size_t jj = 0; jj < 8; jj++) { f.coef.push_back(at(top << 4 | jj)); f.coef.push_back(at(top << 4 | (jj + 8))); }
          double l1 = 0.0;                                             // exact: dyadic numbers of a few bits
          for (size_t si = 0; si < ninner; si++) { l1 += std::fabs(at(si)); if (at(si) != 0.0) f.nonzero++; }
          if (kd >= 3) { f.coef.push_back(l1); f.coef.push_back(0.0); }  // closing unit of the block: (sum |c|, -) for the round-off bound
          f.n_coef += (int64_t)ninner;
        }
        any = f.nonzero > 0;
        if (!any) continue;
        for (int s : ji.pairedSlots) f.paired.push_back((uint8_t)s);
        for (int b = 0; b < kd; b++) f.inner.push_back((uint8_t)ji.binSlots[ko + b]);
        for (int b = 0; b < ko; b++) if (so >> b & 1) f.scal.push_back((uint8_t)(MQ_SC_R << 4 | ji.binSlots[b]));
        for (int s : ji.atSlots) f.scal.push_back((uint8_t)(MQ_SC_AT << 4 | s));
        if (ji.qSlot >= 0) f.scal.push_back((uint8_t)(MQ_SC_AQ << 4 | ji.qSlot));
        famsOf[j].push_back(std::move(f));
      }
  });
  for (auto &v : famsOf) for (auto &f : v) { tb.n_stored += f.n_coef; tb.n_nonzero += f.nonzero; tb.fams.push_back(std::move(f)); }
  lap("families");
  return tb;
}

}  // namespace mq
