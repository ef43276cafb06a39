// fg_plan.cpp — host planner (see fg_plan.hpp).  All citations: PAPER.md = /root/reference/PAPER.md.
//
// What is built here, in the paper's order:
//   graph validity (1PI, no lepton loops)
//   UV-divergent subgraphs: self-energy (N_e=2,N_gamma=0), vertexlike (N_e=2,N_gamma=1)   PAPER.md:139, fn.7
//   forests F[G] and the chain I[G]
//   operator table of R^new: A on G', U below, L above, (L-U) on G     PAPER.md:184-198, example (11) at 200-203
//   per element: loop basis, slot string, Dirac traces of the projectors A, U, L
//   Hepp-sector density tables Deg(s), Z(s)
// The numerator of every (element, operator) is flattened into a stream of "records"
//   value = prod_f V[f] * sum_{T subset of k free slots} coef[T] prod_{j in T} A_j
// that the CUDA kernel interprets.
#include "fg_plan.hpp"

#include <algorithm>
#include <chrono>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <map>
#include <numeric>

#ifdef _OPENMP
#include <omp.h>
#endif

#include "../../include/fg.h"

namespace fg {

// ------------------------------------------------------------------------------------------------
// graph
// ------------------------------------------------------------------------------------------------
static bool spanned(const Graph& g, int lo, int hi, int i) {   // electron line e_i spanned by a photon inside [lo,hi]
  for (auto& p : g.ph) if (p[0] >= lo && p[1] <= hi && p[0] <= i - 1 && p[1] >= i) return true;
  return false;
}

int graph_from_edges(const int32_t* edges, int n_edges, int ext_vertex, Graph& g, std::string& msg) {
  if (!edges || n_edges <= 0) { msg = "no edges"; return FG_E_ARG; }
  if (n_edges % 3 != 0) { msg = "need 3n internal lines"; return FG_E_COUNT; }
  int n = n_edges / 3;
  if (n > FG_MAXL) { msg = "more than 5 loops"; return FG_E_LOOPS; }
  int nv = 2 * n + 1;
  std::vector<std::array<int, 2>> el, pl;
  for (int k = 0; k < n_edges; ++k) {
    int u = edges[3 * k], v = edges[3 * k + 1], kind = edges[3 * k + 2];
    if (u < 0 || v < 0 || u >= nv || v >= nv || u == v) { msg = "vertex out of range (need vertices 0..2n)"; return FG_E_COUNT; }
    if (kind == 0) el.push_back({u, v}); else if (kind == 1) pl.push_back({u, v}); else { msg = "edge kind must be 0 or 1"; return FG_E_ARG; }
  }
  if ((int)el.size() != 2 * n || (int)pl.size() != n) { msg = "need 2n electron and n photon lines"; return FG_E_COUNT; }
  if (ext_vertex < 0 || ext_vertex >= nv) { msg = "external-photon vertex out of range"; return FG_E_ARG; }
  // electron lines must form one open path; follow it u -> v
  std::vector<int> out(nv, -1), indeg(nv, 0), outdeg(nv, 0);
  for (auto& e : el) { if (out[e[0]] >= 0) { msg = "two electron lines leave one vertex"; return FG_E_NOT_PATH; } out[e[0]] = e[1]; ++outdeg[e[0]]; ++indeg[e[1]]; }
  int start = -1;
  for (int v = 0; v < nv; ++v) { if (indeg[v] > 1) { msg = "two electron lines enter one vertex"; return FG_E_NOT_PATH; } if (indeg[v] == 0) { if (start >= 0) { msg = "electron lines are not one path"; return FG_E_NOT_PATH; } start = v; } }
  if (start < 0) { msg = "electron lines close a loop (lepton loop)"; return FG_E_NOT_PATH; }
  std::vector<int> pos(nv, -1); int cur = start, cnt = 0;
  while (cur >= 0 && pos[cur] < 0) { pos[cur] = cnt++; cur = out[cur]; }
  if (cnt != nv) { msg = "electron lines are not one open path through all vertices"; return FG_E_NOT_PATH; }
  g = Graph(); g.n = n; g.nv = nv; g.x = pos[ext_vertex]; g.partner.assign(nv, -1);
  std::vector<int> used(nv, 0); used[g.x] = 1;
  for (auto& p : pl) {
    int a = pos[p[0]], b = pos[p[1]]; if (a > b) std::swap(a, b);
    if (used[a] || used[b]) { msg = "a vertex carries more than one photon"; return FG_E_VERTEX; }
    used[a] = used[b] = 1; g.partner[a] = b; g.partner[b] = a; g.ph.push_back({a, b});
  }
  for (int v = 0; v < nv; ++v) if (!used[v]) { msg = "a vertex carries no photon"; return FG_E_VERTEX; }
  std::sort(g.ph.begin(), g.ph.end());
  for (int i = 1; i <= 2 * n; ++i) if (!spanned(g, 0, 2 * n, i)) { msg = "electron line e_" + std::to_string(i) + " is not spanned by a photon"; return FG_E_NOT_1PI; }
  return FG_OK;
}

// ------------------------------------------------------------------------------------------------
// UV-divergent subgraphs (fn.7 at 155): with no lepton loops each is the induced subgraph on a
// vertex interval whose electron lines are all spanned by internal photons; the number of vertices whose photon
// leaves the interval (v_x counts) is 0 (self-energy) or 1 (vertexlike).
// ------------------------------------------------------------------------------------------------
static bool classify(const Graph& g, int a, int b, Sub& s) {
  int leaving = 0, inside = 0;
  for (int v = a; v <= b; ++v) { int p = g.partner[v]; if (p < 0 || p < a || p > b) ++leaving; else ++inside; }
  if (inside < 2 || leaving > 1) return false;
  for (int i = a + 1; i <= b; ++i) if (!spanned(g, a, b, i)) return false;
  s.a = a; s.b = b; s.type = leaving; s.chain = (leaving == 1 && g.x >= a && g.x <= b);
  return true;
}
static bool contains(const Sub& p, const Sub& q) { return p.a <= q.a && q.b <= p.b; }
static bool overlap(const Sub& p, const Sub& q) {   // share a line, neither contains the other
  return std::max(p.a, q.a) < std::min(p.b, q.b) && !contains(p, q) && !contains(q, p);
}

// ------------------------------------------------------------------------------------------------
// Clifford monomials: s * gamma^mask, gamma^mask = ascending product; {g^mu,g^nu} = 2 diag(+,-,-,-)
// ------------------------------------------------------------------------------------------------
struct CliffTab {
  uint8_t flip[16][4];   // sign flip when gamma^mu is multiplied on the right of gamma^mask
  uint8_t parsp[16];     // parity of the number of spatial gammas = parity of popcount(mask & 0b1110)
  CliffTab() {
    for (int m = 0; m < 16; ++m) {
      parsp[m] = __builtin_popcount(m & 14) & 1;
      for (int mu = 0; mu < 4; ++mu) {
        int f = __builtin_popcount(m >> (mu + 1)) & 1;      // hop over the gammas with larger index
        if (((m >> mu) & 1) && mu != 0) f ^= 1;             // gamma^i gamma^i = -1
        flip[m][mu] = (uint8_t)f;
      }
    }
  }
};
static const CliffTab CT;

static int trace_of(const std::vector<int>& F, int p0, int mask) {   // Tr[ prod F * gamma0^p0 * gamma^mask ]
  int s = 0, m = 0;
  auto mul = [&](int mu) { s ^= CT.flip[m][mu]; m ^= (1 << mu); };
  for (int mu : F) mul(mu);
  if (p0) mul(0);
  for (int mu = 0; mu < 4; ++mu) if ((mask >> mu) & 1) mul(mu);
  return m == 0 ? (s ? -4 : 4) : 0;
}

// One run: sum over the Lorentz indices of all chords (photon chords and Wick pairs) of the signed monomial of the
// string, resolved by the parity pattern `cb` that a gamma^0 placed at each gap would pick up when moved to the front.
struct DiracRun {
  int ntok = 0;
  int8_t kind[48];   // 0 first end of chord, 1 second end, 2 fixed gamma, 3 gap
  int8_t arg[48];
  int8_t val[16];
  int64_t* N = nullptr;
  void go(int pos, unsigned sgn, unsigned mask, unsigned cb) {
    for (;;) {
      if (pos == ntok) { N[cb] += sgn ? -1 : 1; return; }
      int a = arg[pos];
      switch (kind[pos]) {
        case 0:
          for (int mu = 0; mu < 4; ++mu) { val[a] = (int8_t)mu; go(pos + 1, sgn ^ CT.flip[mask][mu], mask ^ (1u << mu), cb); }
          return;
        case 1: { int mu = val[a]; sgn ^= CT.flip[mask][mu] ^ (mu != 0 ? 1u : 0u); mask ^= (1u << mu); break; }   // gamma_rho = g_rr gamma^rho
        case 2: sgn ^= CT.flip[mask][a]; mask ^= (1u << a); break;
        default: cb |= (unsigned)CT.parsp[mask] << a; break;
      }
      ++pos;
    }
  }
};

struct Piece { double w; std::vector<int> F; int ext; bool q; };

static std::vector<Piece> pieces_of(int op, int type, int comp) {
  // Rest frame p = (1,0,0,0), p^2 = m^2 = 1.
  std::vector<Piece> P;
  if (type == 0) {                       // U on a self-energy Sigma = u + v p-hat: u = Tr[Sigma]/4, v = Tr[g0 Sigma]/4
    if (comp == 0) P.push_back({0.25, {}, -1, false}); else P.push_back({0.25, {0}, -1, false});
    return P;
  }
  // Gamma_mu(p,0) = a g_mu + b p_mu + c p-hat p_mu + d(p-hat g_mu - g_mu p-hat)   (10)
  auto addU = [&](double s) { P.push_back({-0.25 * s, {3}, 3, false}); };                      // a = Tr[g^3 Gamma_3]/4, Gamma_3 = -Gamma^3
  auto addL = [&](double s) { P.push_back({0.25 * s, {}, 0, false}); P.push_back({0.25 * s, {0}, 0, false}); };   // a+b+c = Tr[(1+g0)Gamma_0]/4
  if (op == FG_OP_U) addU(1);
  else if (op == FG_OP_L) addL(1);
  else if (op == FG_OP_LMU) { addL(1); addU(-1); }
  else {
    // A: Pauli form factor at q = 0 from Gamma^mu = V^mu + q_nu T^{nu mu}:
    //   (1/12) Tr[g_mu V^mu - (4 g0 + 3) V^0]  =  -(1/4) { Tr[g0 V^0] + Tr[g3 V^3] + Tr[V^0] }   (isotropy)
    //   (1/48) sum_{mu != nu} Tr[(g0+1)[g_mu,g_nu](g0+1) T^{nu mu}] = (1/2) Tr[g1 g2 (1+g0) T^{21}]
    P.push_back({-0.25, {0}, 0, false}); P.push_back({-0.25, {3}, 3, false}); P.push_back({-0.25, {}, 0, false});
    P.push_back({0.5, {1, 2}, 1, true}); P.push_back({0.5, {1, 2, 0}, 1, true});
  }
  return P;
}

// ------------------------------------------------------------------------------------------------
// element geometry
// ------------------------------------------------------------------------------------------------
static HGeom make_geom(const Graph& g, const std::vector<Sub>& subs, int si, const std::vector<int>& kids) {
  HGeom E; E.sub = si; E.kids = kids;
  const Sub& S = subs[si];
  int n2 = 2 * g.n;
  struct Site { int kind, v, kid; };   // kind 0 plain vertex, 1 vertexlike child, 2 self-energy child
  std::vector<Site> sites; std::vector<int> site_of(g.nv, -1);
  for (int v = S.a; v <= S.b; ++v) {
    int kid = -1; for (int c : kids) if (subs[c].a == v) kid = c;
    int s = (int)sites.size();
    if (kid >= 0) { sites.push_back({subs[kid].type == 1 ? 1 : 2, v, kid}); for (int w = subs[kid].a; w <= subs[kid].b; ++w) site_of[w] = s; v = subs[kid].b; }
    else { sites.push_back({0, v, -1}); site_of[v] = s; }
    if (v < S.b) E.own_e.push_back(v);   // line e_{v+1} = (v_v, v_{v+1}) has id v; it joins site s and site s+1
  }
  E.ne = (int)E.own_e.size();
  std::vector<int> chord(g.n, -1); std::vector<std::array<int, 2>> ph_sites;
  for (int k = 0; k < g.n; ++k) {
    int a = g.ph[k][0], b = g.ph[k][1];
    if (a < S.a || b > S.b || site_of[a] == site_of[b]) continue;
    chord[k] = (int)E.own_ph.size(); E.own_ph.push_back(n2 + k); ph_sites.push_back({site_of[a], site_of[b]});
  }
  E.l = (int)E.own_ph.size();
  E.eta.assign(E.ne, 0);
  for (int q = 0; q < E.ne; ++q) for (int a = 0; a < E.l; ++a) if (ph_sites[a][0] <= q && q < ph_sites[a][1]) E.eta[q] |= (1 << a);
  E.has_x = (g.x >= S.a && g.x <= S.b);
  int xsite = E.has_x ? site_of[g.x] : -1;
  E.xiq.assign(E.ne, 0);
  if (E.has_x) for (int q = 0; q < E.ne; ++q) E.xiq[q] = (q + 1 <= xsite) ? -1 : +1;
  int ext_site = -1;
  if (S.type == 1) for (int w = S.a; w <= S.b; ++w) { int p = g.partner[w]; if (p < 0 || p < S.a || p > S.b) ext_site = site_of[w]; }
  for (auto& st : sites) { if (st.kind == 2) E.se_kids.push_back(st.kid); if (st.kind == 1) E.vc_kids.push_back(st.kid); }
  // tokens in path order: site, line, site, ...; reversed below (the matrix string reads from v_b back to v_a)
  std::vector<Tok> fw; std::vector<Slot> fslots;
  for (int s = 0; s < (int)sites.size(); ++s) {
    const Site& st = sites[s];
    if (st.kind == 2) {
      int idx = (int)(std::find(E.se_kids.begin(), E.se_kids.end(), st.kid) - E.se_kids.begin());
      fw.push_back({2, (int)fslots.size()}); fslots.push_back({s - 1, idx, E.has_x ? (s < xsite ? -1 : +1) : 0});
    } else if (s == ext_site) fw.push_back({1, 0});
    else {
      int k = -1;   // the photon attached here: a plain vertex's own photon, or the one photon leaving a vertexlike child
      for (int q = 0; q < g.n; ++q) {
        if (st.kind == 0) { if (g.ph[q][0] == st.v || g.ph[q][1] == st.v) k = q; }
        else { const Sub& K = subs[st.kid]; bool ia = g.ph[q][0] >= K.a && g.ph[q][0] <= K.b, ib = g.ph[q][1] >= K.a && g.ph[q][1] <= K.b; if (ia != ib) k = q; }
      }
      fw.push_back({0, chord[k]});
    }
    if (s + 1 < (int)sites.size()) { fw.push_back({2, (int)fslots.size()}); fslots.push_back({s, -1, E.xiq[s]}); }
  }
  int ns = (int)fslots.size();
  for (int i = (int)fw.size() - 1; i >= 0; --i) { Tok t = fw[i]; if (t.kind == 2) t.id = ns - 1 - t.id; E.toks.push_back(t); }
  E.slots.assign(fslots.rbegin(), fslots.rend());
  return E;
}

// ------------------------------------------------------------------------------------------------
// numerator records of one (geometry, operator)
// ------------------------------------------------------------------------------------------------
struct Matching { std::vector<std::array<int, 2>> pairs; std::vector<int> unmatched; };
static void enum_matchings(int ns, std::vector<Matching>& out) {
  std::vector<int> used(ns, 0); Matching cur;
  struct R { static void go(int i, int ns, std::vector<int>& used, Matching& cur, std::vector<Matching>& out) {
    while (i < ns && used[i]) ++i;
    if (i == ns) { out.push_back(cur); return; }
    used[i] = 1;
    cur.unmatched.push_back(i); go(i + 1, ns, used, cur, out); cur.unmatched.pop_back();
    for (int j = i + 1; j < ns; ++j) if (!used[j]) { used[j] = 1; cur.pairs.push_back({i, j}); go(i + 1, ns, used, cur, out); cur.pairs.pop_back(); used[j] = 0; }
    used[i] = 0;
  } };
  R::go(0, ns, used, cur, out);
  for (auto& m : out) std::sort(m.unmatched.begin(), m.unmatched.end());
}

// table over subsets T of `gaps` (bit g of T = gaps[g] carries gamma^0) of the coefficient of this matching
static void matching_table(const HGeom& E, int type, int op, int comp, const Matching& m, int qslot, bool qpart,
                           const std::vector<int>& gaps, std::vector<double>& out) {
  int ng = (int)gaps.size(); size_t nT = (size_t)1 << ng;
  out.assign(nT, 0.0);
  std::vector<Piece> pcs = pieces_of(op, type, comp);
  std::vector<int> exts;
  for (auto& p : pcs) if (p.q == qpart && std::find(exts.begin(), exts.end(), p.ext) == exts.end()) exts.push_back(p.ext);
  int ns = (int)E.slots.size();
  std::vector<int> role(ns, -1), gapidx(ns, -1);
  for (size_t k = 0; k < m.pairs.size(); ++k) { role[m.pairs[k][0]] = (int)k; role[m.pairs[k][1]] = (int)k; }
  for (int gi = 0; gi < ng; ++gi) gapidx[gaps[gi]] = gi;
  const int NU = 2;
  std::vector<int64_t> N(nT);
  for (int ext : exts) {
    DiracRun R; R.N = N.data(); std::fill(N.begin(), N.end(), 0);
    std::vector<int> seen(E.l + m.pairs.size(), 0);
    int fm = 0;
    for (const Tok& t : E.toks) {
      int chord = -1;
      if (t.kind == 1) { R.kind[R.ntok] = 2; R.arg[R.ntok++] = (int8_t)ext; fm ^= (1 << ext); continue; }
      if (t.kind == 0) chord = t.id;
      else if (t.id == qslot) { R.kind[R.ntok] = 2; R.arg[R.ntok++] = NU; fm ^= (1 << NU); continue; }
      else if (role[t.id] < 0) { R.kind[R.ntok] = 3; R.arg[R.ntok++] = (int8_t)gapidx[t.id]; continue; }
      else chord = E.l + role[t.id];
      R.kind[R.ntok] = (int8_t)(seen[chord] ? 1 : 0); R.arg[R.ntok++] = (int8_t)chord; seen[chord] = 1;
    }
    R.go(0, 0u, 0u, 0u);
    // Walsh-Hadamard: H[T] = sum_cb N[cb] (-1)^{|T & cb|}
    for (size_t h = 1; h < nT; h <<= 1) for (size_t i = 0; i < nT; i += (h << 1)) for (size_t j = i; j < i + h; ++j) { int64_t a = N[j], b = N[j + h]; N[j] = a + b; N[j + h] = a - b; }
    for (auto& p : pcs) if (p.q == qpart && p.ext == ext) {
      int tr[2] = {trace_of(p.F, 0, fm), trace_of(p.F, 1, fm)};
      for (size_t T = 0; T < nT; ++T) { int t = tr[__builtin_popcountll(T) & 1]; if (t) out[T] += p.w * (double)t * (double)N[T]; }
    }
  }
  double pref = 1.0; for (size_t k = 0; k < m.pairs.size(); ++k) pref *= -0.5;   // <kappa_i^mu kappa_j^nu> = -(1/2) beta_ij g^{mu nu} t
  for (auto& c : out) c *= pref;
}

static void finish_record(HRecord& r) {
  r.cabs[0] = r.cabs[1] = 0.f;
  if (r.flags & FG_REC_TWO) { size_t h = (size_t)1 << r.k; double a0 = 0, a1 = 0; for (size_t i = 0; i < h; ++i) { a0 += std::fabs(r.coef[i]); a1 += std::fabs(r.coef[h + i]); } r.cabs[0] = (float)(a0 * 1.0000002); r.cabs[1] = (float)(a1 * 1.0000002); }
  else { double a0 = 0; for (double v : r.coef) a0 += std::fabs(v); r.cabs[0] = (float)(a0 * 1.0000002); }
  if (r.coef.size() & 1) r.coef.push_back(0.0);
}

static void build_records(const HGeom& E, int type, HNum& N, bool& limit_hit) {
  int ns = (int)E.slots.size(), ne = E.ne, nb = ne * (ne + 1) / 2;
  auto bidx = [&](int i, int j) { if (i > j) std::swap(i, j); return i * ne - i * (i - 1) / 2 + (j - i); };
  std::vector<Matching> ms; enum_matchings(ns, ms);
  std::vector<std::vector<HRecord>> per(ms.size());
  int ncomp = N.ncomp; bool over = false;
#pragma omp parallel for schedule(dynamic, 1)
  for (long mi = 0; mi < (long)ms.size(); ++mi) {
    const Matching& m = ms[mi];
    int npairs = (int)m.pairs.size();
    int sig0 = 0; std::vector<int> f0;
    for (auto& pr : m.pairs) { f0.push_back(bidx(E.slots[pr[0]].e, E.slots[pr[1]].e)); for (int t = 0; t < 2; ++t) if (E.slots[pr[t]].se >= 0) sig0 |= 1 << E.slots[pr[t]].se; }
    bool wantq = (N.op == FG_OP_A && type == 1);
    bool pseudo = false; for (int s : m.unmatched) if (E.slots[s].se >= 0) pseudo = true;
    int k = (int)m.unmatched.size();
    if (wantq) {
      // Operator A: besides the gamma^0 A_j terms exactly one unmatched slot may carry gamma^nu A^q_j.
      // Free variables of the records = the first FG_KMAX unmatched OWN lines; every other unmatched slot (further own
      // lines, pseudo-slots of self-energy children) is enumerated: in the set -> product factor A_j (and the v
      // component of the child), not in the set -> factor 1 (u component).  The gamma^nu slot is either a free variable
      // (q-extension tables of the same record) or an enumerated slot (own records with the factor A^q).
      const std::vector<int>& um = m.unmatched;
      std::vector<int> mat, en;
      for (int sl : um) { if (E.slots[sl].se < 0 && (int)mat.size() < FG_KMAX) mat.push_back(sl); else en.push_back(sl); }
      const int km = (int)mat.size(), ke = (int)en.size();
      if (npairs + ke + 1 > FG_MAXF) { over = true; continue; }
      auto tab_index = [](const std::vector<int>& gaps, const std::vector<int>& set) { size_t T = 0; for (int sl : set) { size_t pos = std::find(gaps.begin(), gaps.end(), sl) - gaps.begin(); T |= (size_t)1 << pos; } return T; };
      std::vector<double> main_t; matching_table(E, type, N.op, 0, m, -1, false, um, main_t);
      std::vector<std::vector<double>> qt(k); std::vector<std::vector<int>> qgaps(k);
      for (int j = 0; j < k; ++j) { for (int sl : um) if (sl != um[j]) qgaps[j].push_back(sl); matching_table(E, type, N.op, 0, m, um[j], true, qgaps[j], qt[j]); }
      auto pos_in_um = [&](int sl) { return (int)(std::find(um.begin(), um.end(), sl) - um.begin()); };
      auto fill_common = [&](HRecord& r, const std::vector<int>& extra, int sig) {
        std::memset(r.fidx, 0, sizeof(r.fidx)); std::memset(r.vidx, 0, sizeof(r.vidx));
        std::vector<int> f = f0; for (int v : extra) f.push_back(v);
        r.nf = (int)f.size(); for (int t = 0; t < r.nf; ++t) r.fidx[t] = (uint8_t)f[t];
        r.k = km; for (int t = 0; t < km; ++t) r.vidx[t] = (uint8_t)(nb + E.slots[mat[t]].e);
        r.dst = sig * FG_NDEG + npairs;
      };
      for (unsigned eb = 0; eb < (1u << ke); ++eb) {
        std::vector<int> te, extra; int sig = sig0;
        for (int t = 0; t < ke; ++t) if ((eb >> t) & 1) { const Slot& sl = E.slots[en[t]]; te.push_back(en[t]); extra.push_back(nb + sl.e); if (sl.se >= 0) sig |= 1 << sl.se; }
        HRecord r; r.flags = 0; fill_common(r, extra, sig);
        r.coef.assign((size_t)1 << km, 0.0); bool nz = false, nzq = false;
        for (size_t sub = 0; sub < ((size_t)1 << km); ++sub) {
          std::vector<int> set = te; for (int t = 0; t < km; ++t) if ((sub >> t) & 1) set.push_back(mat[t]);
          double v = main_t[tab_index(um, set)]; r.coef[sub] = v; if (v != 0.0) nz = true;
        }
        std::vector<double> qall;
        for (int j = 0; j < km; ++j) {
          const int ju = pos_in_um(mat[j]);
          std::vector<int> rest; for (int t = 0; t < km; ++t) if (t != j) rest.push_back(mat[t]);
          for (size_t sub = 0; sub < ((size_t)1 << (km - 1)); ++sub) {
            std::vector<int> set = te; for (int t = 0; t < km - 1; ++t) if ((sub >> t) & 1) set.push_back(rest[t]);
            double v = qt[ju][tab_index(qgaps[ju], set)]; qall.push_back(v); if (v != 0.0) nzq = true;
          }
        }
        if (nzq) { r.flags |= FG_REC_QEXT; r.coef.insert(r.coef.end(), qall.begin(), qall.end()); }
        if (nz || nzq) { finish_record(r); per[mi].push_back(std::move(r)); }
      }
      for (int jq = 0; jq < ke; ++jq) {       // gamma^nu on an enumerated slot
        const Slot& qs = E.slots[en[jq]]; const int ju = pos_in_um(en[jq]);
        std::vector<int> others; for (int t = 0; t < ke; ++t) if (t != jq) others.push_back(en[t]);
        for (unsigned eb = 0; eb < (1u << others.size()); ++eb) {
          std::vector<int> te, extra = {nb + ne + qs.e}; int sig = sig0 | (qs.se >= 0 ? 1 << qs.se : 0);
          for (size_t t = 0; t < others.size(); ++t) if ((eb >> t) & 1) { const Slot& sl = E.slots[others[t]]; te.push_back(others[t]); extra.push_back(nb + sl.e); if (sl.se >= 0) sig |= 1 << sl.se; }
          HRecord r; r.flags = 0; fill_common(r, extra, sig);
          r.coef.assign((size_t)1 << km, 0.0); bool nz = false;
          for (size_t sub = 0; sub < ((size_t)1 << km); ++sub) {
            std::vector<int> set = te; for (int t = 0; t < km; ++t) if ((sub >> t) & 1) set.push_back(mat[t]);
            double v = qt[ju][tab_index(qgaps[ju], set)]; r.coef[sub] = v; if (v != 0.0) nz = true;
          }
          if (nz) { finish_record(r); per[mi].push_back(std::move(r)); }
        }
      }
      continue;
    }
    std::vector<int> qchoices = {-1};
    if (wantq) for (int s : m.unmatched) qchoices.push_back(s);
    for (int q : qchoices) {
      std::vector<int> gaps; for (int s : m.unmatched) if (s != q) gaps.push_back(s);
      std::vector<double> tab[2];
      for (int c = 0; c < ncomp; ++c) matching_table(E, type, N.op, c, m, q, q >= 0, gaps, tab[c]);
      bool any = false; for (int c = 0; c < ncomp; ++c) for (double v : tab[c]) if (v != 0.0) any = true;
      if (!any) continue;
      // split the gaps: pseudo-slots (self-energy children) and own lines beyond FG_KMAX are enumerated
      std::vector<int> en, fr;   // positions in `gaps`
      for (int gi = 0; gi < (int)gaps.size(); ++gi) { if (E.slots[gaps[gi]].se >= 0) en.push_back(gi); else fr.push_back(gi); }
      while ((int)fr.size() > FG_KMAX) { en.push_back(fr.back()); fr.pop_back(); }
      int sigq = sig0; std::vector<int> fq = f0;
      if (q >= 0) { fq.push_back(nb + ne + E.slots[q].e); if (E.slots[q].se >= 0) sigq |= 1 << E.slots[q].se; }
      for (unsigned eb = 0; eb < (1u << en.size()); ++eb) {
        HRecord r; r.flags = (ncomp == 2) ? FG_REC_TWO : 0; r.k = (int)fr.size(); int sig = sigq; std::vector<int> f = fq; size_t Tbase = 0;
        for (size_t t = 0; t < en.size(); ++t) if ((eb >> t) & 1) { const Slot& sl = E.slots[gaps[en[t]]]; f.push_back(nb + sl.e); if (sl.se >= 0) sig |= 1 << sl.se; Tbase |= (size_t)1 << en[t]; }
        if ((int)f.size() > FG_MAXF) { over = true; continue; }
        r.nf = (int)f.size(); r.dst = sig * FG_NDEG + npairs;
        std::memset(r.fidx, 0, sizeof(r.fidx)); std::memset(r.vidx, 0, sizeof(r.vidx));
        for (int t = 0; t < r.nf; ++t) r.fidx[t] = (uint8_t)f[t];
        for (int t = 0; t < r.k; ++t) r.vidx[t] = (uint8_t)(nb + E.slots[gaps[fr[t]]].e);
        r.coef.assign((size_t)ncomp << r.k, 0.0); bool nz = false;
        for (int c = 0; c < ncomp; ++c) for (size_t sub = 0; sub < ((size_t)1 << r.k); ++sub) {
          size_t T = Tbase; for (int t = 0; t < r.k; ++t) if ((sub >> t) & 1) T |= (size_t)1 << fr[t];
          double v = tab[c][T]; r.coef[((size_t)c << r.k) + sub] = v; if (v != 0.0) nz = true;
        }
        if (nz) { finish_record(r); per[mi].push_back(std::move(r)); }
      }
    }
  }
  if (over) limit_hit = true;
  for (auto& v : per) for (auto& r : v) N.recs.push_back(std::move(r));
  std::stable_sort(N.recs.begin(), N.recs.end(), [](const HRecord& a, const HRecord& b) {
    if (a.dst != b.dst) return a.dst < b.dst;
    if (a.nf != b.nf) return a.nf < b.nf;
    if (a.k != b.k) return a.k > b.k;
    if ((a.flags & 3) != (b.flags & 3)) return (a.flags & 3) < (b.flags & 3);
    return std::memcmp(a.vidx, b.vidx, sizeof(a.vidx)) < 0; });
  for (auto& r : N.recs) {
    long nc = (long)r.coef.size(), nz = 0; for (double v : r.coef) if (v != 0.0) ++nz;
    int nco = (r.flags & FG_REC_TWO) ? 2 : 1;
    N.n_coefs += nc; N.n_nonzero += nz;
    N.algo_flops += 2.0 * nz;
  }
}

// Debug surface (fg_host_dirac_table): the coefficient table of ONE matching of ONE element, straight from matching_table.
int dirac_table(const Graph& g, int a, int b, const std::vector<std::array<int, 2>>& kid_iv, int op, int comp,
                const std::vector<std::array<int, 2>>& pairs, int qslot, std::vector<double>& table, std::vector<int>& gaps, std::string& msg) {
  std::vector<Sub> subs; Sub S;
  if (!classify(g, a, b, S)) { msg = "[a,b] is not a UV-divergent subgraph"; return FG_E_ARG; }
  subs.push_back(S); std::vector<int> kids;
  for (auto& iv : kid_iv) { Sub K; if (!classify(g, iv[0], iv[1], K) || !contains(S, K)) { msg = "child interval is not a UV-divergent subgraph inside [a,b]"; return FG_E_ARG; } kids.push_back((int)subs.size()); subs.push_back(K); }
  HGeom E = make_geom(g, subs, 0, kids);
  const int ns = (int)E.slots.size();
  Matching m; std::vector<int> used(ns, 0);
  for (auto& pr : pairs) { if (pr[0] < 0 || pr[1] >= ns || pr[0] >= pr[1] || used[pr[0]] || used[pr[1]]) { msg = "bad pair"; return FG_E_ARG; } used[pr[0]] = used[pr[1]] = 1; m.pairs.push_back(pr); }
  for (int sl = 0; sl < ns; ++sl) if (!used[sl]) m.unmatched.push_back(sl);
  if (qslot >= 0 && (qslot >= ns || used[qslot])) { msg = "bad q slot"; return FG_E_ARG; }
  gaps.clear(); for (int sl : m.unmatched) if (sl != qslot) gaps.push_back(sl);
  matching_table(E, S.type, op, comp, m, qslot, qslot >= 0, gaps, table);
  return ns;
}

// ------------------------------------------------------------------------------------------------
// density tables.  Deg(s): the paper's algorithm (constants (15)) is only in
// its Refs. [42],[32]; reading R-Deg is used unless the caller supplies a table.
// ------------------------------------------------------------------------------------------------
static void build_density(HostPlan& P) {
  const Graph& g = P.g; int n = g.n, M = P.M; size_t nset = (size_t)1 << M;
  P.deg.assign(nset, 0.0);
  if (!P.opts.deg_override.empty()) { for (size_t s = 1; s + 1 < nset; ++s) P.deg[s] = P.opts.deg_override[s]; }
  else {
    for (size_t s = 1; s + 1 < nset; ++s) {
      std::vector<char> in(3 * n, 0);
      for (int v = 0; v < M; ++v) if ((s >> v) & 1) for (int id : P.var_lines[v]) in[id] = 1;
      std::vector<int> root(g.nv); std::iota(root.begin(), root.end(), 0);
      auto find = [&](int a) { while (root[a] != a) a = root[a] = root[root[a]]; return a; };
      int ne = 0, np = 0, indep = 0;
      for (int id = 0; id < 3 * n; ++id) if (in[id]) {
        int a = id < 2 * n ? id : g.ph[id - 2 * n][0], b = id < 2 * n ? id + 1 : g.ph[id - 2 * n][1];
        (id < 2 * n ? ne : np)++;
        int ra = find(a), rb = find(b); if (ra != rb) { root[ra] = rb; ++indep; }
      }
      int loops = ne + np - indep;
      double omega = 2.0 * loops - 0.5 * ne - 1.0 * np;          // superficial degree of the line set
      std::vector<int> inside;
      for (size_t k = 1; k < P.subs.size(); ++k) {
        const Sub& S = P.subs[k]; bool all = true;
        for (int i = S.a; i < S.b; ++i) if (!in[i]) all = false;
        for (int q = 0; q < n; ++q) if (g.ph[q][0] >= S.a && g.ph[q][1] <= S.b && !in[2 * n + q]) all = false;
        if (all) inside.push_back((int)k);
      }
      for (int k : inside) {
        bool maximal = true; for (int k2 : inside) if (k2 != k && contains(P.subs[k2], P.subs[k])) maximal = false;
        if (maximal) omega -= (P.subs[k].type == 1 ? 0.0 : 0.5) + 0.5;   // remove omega(S) + 1/2 of a subtracted subgraph
      }
      P.deg[s] = std::min(1.5, std::max(0.5, -omega));
    }
  }
  auto buildZ = [&](double scale, std::vector<double>& Z) {
    Z.assign(nset, 0.0); Z[0] = 1.0;
    for (size_t s = 1; s < nset; ++s) {
      double sum = 0.0;
      for (int j = 0; j < M; ++j) if ((s >> j) & 1) sum = sum + Z[s ^ ((size_t)1 << j)];
      Z[s] = (s + 1 < nset) ? sum / (scale * P.deg[s]) : sum;
    }
  };
  buildZ(1.0, P.Z1); buildZ(P.opts.D, P.Z3);
  P.lnZfull[0] = std::log(P.Z1[nset - 1]); P.lnZfull[2] = std::log(P.Z3[nset - 1]);
  double lz = 0.0; for (int k = 1; k < M; ++k) lz += std::log(2.0 * k);   // Deg = 1/2: Z(s) = 2^|s| |s|!
  P.lnZfull[1] = lz + std::log((double)M); P.lnZfull[3] = std::log((double)M);   // Deg = |s|: Z = 1
}

// ------------------------------------------------------------------------------------------------
// the plan
// ------------------------------------------------------------------------------------------------
int build_plan(const Graph& g, const PlanOpts& opts, HostPlan& P, std::string& msg) {
  auto t0 = std::chrono::steady_clock::now();
  P = HostPlan(); P.g = g; P.opts = opts;
  int n = g.n;
  double csum = 0; for (int k = 0; k < 4; ++k) { if (!(opts.C[k] >= 0)) { msg = "C_k must be >= 0"; return FG_E_OPTS; } csum += opts.C[k]; }
  if (std::fabs(csum - 1.0) > 1e-12 || !(opts.D > 0)) { msg = "C must sum to 1 and D must be > 0"; return FG_E_OPTS; }
  // variables (the two electron lines at v_x may share one variable)
  for (int id = 0; id < 3 * n; ++id) {
    if (opts.merge && id == g.x - 1) { P.merge_var = (int)P.var_lines.size(); P.var_lines.push_back({g.x - 1, g.x}); }
    else if (opts.merge && id == g.x) continue;
    else P.var_lines.push_back({id});
  }
  P.M = (int)P.var_lines.size();
  if (!opts.deg_override.empty() && opts.deg_override.size() != ((size_t)1 << P.M)) { msg = "deg_table must have 2^M entries"; return FG_E_OPTS; }
  // subgraphs
  Sub G; if (!classify(g, 0, 2 * n, G) || !G.chain) { msg = "graph is not a vertex graph"; return FG_E_NOT_1PI; }
  P.subs.push_back(G);
  for (int a = 0; a <= 2 * n; ++a) for (int b = a + 1; b <= 2 * n; ++b) { if (a == 0 && b == 2 * n) continue; Sub s; if (classify(g, a, b, s)) P.subs.push_back(s); }
  int np = (int)P.subs.size() - 1;
  if (np > 20) { msg = "too many subgraphs"; return FG_E_LIMIT; }
  // forests
  for (uint32_t mask = 0; mask < (1u << np); ++mask) {
    std::vector<int> mem = {0}; bool ok = true;
    for (int i = 0; i < np && ok; ++i) if ((mask >> i) & 1) { for (int j : mem) if (j && overlap(P.subs[i + 1], P.subs[j])) ok = false; mem.push_back(i + 1); }
    if (ok) P.forests.push_back(mem);
  }
  // terms
  for (auto& F : P.forests) {
    if ((int)F.size() > FG_MAXMEM) { msg = "forest too large"; return FG_E_LIMIT; }
    std::vector<int> chain; for (int m : F) if (P.subs[m].chain) chain.push_back(m);
    std::sort(chain.begin(), chain.end(), [&](int p, int q) { return P.subs[p].b - P.subs[p].a > P.subs[q].b - P.subs[q].a; });
    for (size_t r = 0; r < chain.size(); ++r) {
      HTerm t; t.members = F; t.gprime = chain[r]; t.sign = (F.size() % 2 == 1) ? +1 : -1;
      for (int m : F) {
        size_t pos = std::find(chain.begin(), chain.end(), m) - chain.begin();
        int op;
        if (pos == chain.size()) op = FG_OP_U;            // not in I[G]
        else if (pos == r) op = FG_OP_A;                  // G'
        else if (pos > r) op = FG_OP_U;                   // inside G'
        else op = (m == 0) ? FG_OP_LMU : FG_OP_L;         // contains G'
        t.ops.push_back(op);
      }
      P.terms.push_back(t);
    }
  }
  // geometries, programs, nodes
  std::map<std::vector<int>, int> gmap, nmap, ndmap;
  for (auto& t : P.terms) {
    std::map<int, std::vector<int>> kids_of; std::map<int, int> op_of;
    for (size_t k = 0; k < t.members.size(); ++k) {
      int m = t.members[k]; op_of[m] = t.ops[k];
      std::vector<int> ch;
      for (int c : t.members) if (c != m && contains(P.subs[m], P.subs[c])) {
        bool maximal = true;
        for (int d : t.members) if (d != m && d != c && contains(P.subs[d], P.subs[c]) && contains(P.subs[m], P.subs[d])) maximal = false;
        if (maximal) ch.push_back(c);
      }
      std::sort(ch.begin(), ch.end(), [&](int p, int q) { return P.subs[p].a < P.subs[q].a; });
      kids_of[m] = ch;
    }
    std::map<int, int> geom_of;
    struct R { static int go(HostPlan& P, int m, std::map<int, std::vector<int>>& kids_of, std::map<int, int>& op_of, std::map<int, int>& geom_of,
                             std::map<std::vector<int>, int>& gmap, std::map<std::vector<int>, int>& nmap, std::map<std::vector<int>, int>& ndmap) {
      std::vector<int> gk = {m}; for (int c : kids_of[m]) gk.push_back(c);
      int gi; auto it = gmap.find(gk);
      if (it == gmap.end()) { gi = (int)P.geoms.size(); P.geoms.push_back(make_geom(P.g, P.subs, m, kids_of[m])); gmap[gk] = gi; } else gi = it->second;
      geom_of[m] = gi;
      std::vector<int> nk = {gi, op_of[m]}; int ni; auto it2 = nmap.find(nk);
      if (it2 == nmap.end()) { ni = (int)P.nums.size(); HNum N; N.geom = gi; N.op = op_of[m]; N.ncomp = P.subs[m].type == 0 ? 2 : 1; N.nse = (int)P.geoms[gi].se_kids.size(); P.nums.push_back(N); nmap[nk] = ni; } else ni = it2->second;
      HNode nd; nd.num = ni; std::vector<int> key = {ni};
      const std::vector<int> se_kids = P.geoms[gi].se_kids, vc_kids = P.geoms[gi].vc_kids;   // copies: the recursion grows P.geoms
      for (int c : se_kids) { int id = go(P, c, kids_of, op_of, geom_of, gmap, nmap, ndmap); nd.se_kid.push_back(id); key.push_back(id); }
      key.push_back(-1);
      for (int c : vc_kids) { int id = go(P, c, kids_of, op_of, geom_of, gmap, nmap, ndmap); nd.vc_kid.push_back(id); key.push_back(id); }
      auto it3 = ndmap.find(key); if (it3 != ndmap.end()) return it3->second;
      int id = (int)P.nodes.size(); P.nodes.push_back(nd); ndmap[key] = id; return id;
    } };
    t.top = R::go(P, 0, kids_of, op_of, geom_of, gmap, nmap, ndmap);
    for (int m : t.members) t.geoms.push_back(geom_of[m]);
  }
  for (auto& E : P.geoms) if ((int)E.se_kids.size() > FG_MAXSE || (int)E.vc_kids.size() > FG_MAXVC || E.ne > FG_MAXNE || E.l > FG_MAXL) { msg = "element limit exceeded"; return FG_E_LIMIT; }
  // evaluation order: children (shorter intervals) first.  Renumber geoms, nums, nodes accordingly.
  {
    int ng = (int)P.geoms.size();
    std::vector<int> order(ng); std::iota(order.begin(), order.end(), 0);
    std::stable_sort(order.begin(), order.end(), [&](int p, int q) { const Sub& a = P.subs[P.geoms[p].sub]; const Sub& b = P.subs[P.geoms[q].sub]; return a.b - a.a < b.b - b.a; });
    std::vector<int> gnew(ng); std::vector<HGeom> G2; for (int i = 0; i < ng; ++i) { gnew[order[i]] = i; G2.push_back(P.geoms[order[i]]); }
    P.geoms.swap(G2);
    for (auto& N : P.nums) N.geom = gnew[N.geom];
    for (auto& t : P.terms) for (int& q : t.geoms) q = gnew[q];
    int nn = (int)P.nums.size();
    std::vector<int> norder(nn); std::iota(norder.begin(), norder.end(), 0);
    std::stable_sort(norder.begin(), norder.end(), [&](int p, int q) { return P.nums[p].geom < P.nums[q].geom; });
    std::vector<int> nnew(nn); std::vector<HNum> N2; for (int i = 0; i < nn; ++i) { nnew[norder[i]] = i; N2.push_back(P.nums[norder[i]]); }
    P.nums.swap(N2);
    for (auto& nd : P.nodes) nd.num = nnew[nd.num];
    int nd_n = (int)P.nodes.size();
    std::vector<int> dorder(nd_n); std::iota(dorder.begin(), dorder.end(), 0);
    std::stable_sort(dorder.begin(), dorder.end(), [&](int p, int q) { return P.nodes[p].num < P.nodes[q].num; });
    std::vector<int> dnew(nd_n); std::vector<HNode> D2; for (int i = 0; i < nd_n; ++i) { dnew[dorder[i]] = i; D2.push_back(P.nodes[dorder[i]]); }
    P.nodes.swap(D2);
    for (auto& nd : P.nodes) { for (int& k : nd.se_kid) k = dnew[k]; for (int& k : nd.vc_kid) k = dnew[k]; }
    for (auto& t : P.terms) t.top = dnew[t.top];
    for (int i = 0; i < nd_n; ++i) P.nums[P.nodes[i].num].nodes.push_back(i);
  }
  if (opts.structure_only) { build_density(P); P.plan_seconds = std::chrono::duration<double>(std::chrono::steady_clock::now() - t0).count(); return FG_OK; }
  // Dirac tables -> records
  { bool limit_hit = false; for (auto& N : P.nums) build_records(P.geoms[N.geom], P.subs[P.geoms[N.geom].sub].type, N, limit_hit);
    if (limit_hit) { msg = "a numerator record needs more than FG_MAXF product factors"; return FG_E_LIMIT; } }
  // flatten
  P.d_geoms.resize(P.geoms.size());
  for (size_t i = 0; i < P.geoms.size(); ++i) {
    const HGeom& E = P.geoms[i]; FgGeomDev d; std::memset(&d, 0, sizeof(d));
    d.ne = (uint8_t)E.ne; d.l = (uint8_t)E.l; d.has_x = E.has_x;
    for (int q = 0; q < E.ne; ++q) { d.line_e[q] = (uint8_t)E.own_e[q]; d.eta[q] = (uint8_t)E.eta[q]; d.xiq[q] = (int8_t)E.xiq[q]; }
    for (int a = 0; a < E.l; ++a) d.line_ph[a] = (uint8_t)E.own_ph[a];
    P.d_geoms[i] = d;
  }
  P.d_geom_num_begin.assign(P.geoms.size() + 1, 0);
  P.d_geom_voff.clear(); P.vtot = 0; P.vmax = 1;
  for (auto& E : P.geoms) { const int nv = E.ne * (E.ne + 1) / 2 + 2 * E.ne; P.d_geom_voff.push_back(P.vtot); P.vtot += nv; P.vmax = std::max(P.vmax, nv); }
  P.d_geom_voff.push_back(P.vtot);
  int raw_max = 0;
  std::map<std::vector<int>, std::array<long, 3>> hist;   // (mma, nf, k, qx, two) -> records, tiles, groups   (FG_PLAN_HIST=1 prints it)
  for (size_t i = 0; i < P.nums.size(); ++i) {
    HNum& N = P.nums[i]; FgNumDev d; std::memset(&d, 0, sizeof(d));
    d.geom = N.geom; d.op = N.op; d.ncomp = N.ncomp; d.nse = N.nse;
    d.node_begin = N.nodes.empty() ? 0 : N.nodes.front(); d.node_count = (int)N.nodes.size();
    d.chunk_begin = (int)(P.d_chunks.size() / FG_CHUNK_BYTES);
    // pack records into chunks of class-uniform groups; keep = leading product factors shared with the previous record.
    // Runs of records with the same class and the same free variables become tensor-core (DMMA) tile groups.
    size_t cur = 0, base = 0, ghdr = 0; bool open = false, gopen = false; int ngroups = 0, gn = 0; const HRecord* prev = nullptr;
    auto mma_steps = [](int k, bool qx) { if (k < 2) return 1; int nm = 1 << (k - 2); return nm + (qx ? nm + (k - 2) * ((1 << k) >> 3) : 0); };
    auto rec_ncoef_host = [](int k, int flags) { int n = (flags & FG_REC_QEXT) ? (1 << k) + k * ((1 << k) >> 1) : ((flags & FG_REC_TWO) ? 2 : 1) << k; return (n + 1) & ~1; };
    auto cls = [](const HRecord& r) { int fl = r.flags & (FG_REC_TWO | FG_REC_QEXT); if (r.nf > FG_NFC) fl |= FG_REC_WIDE; return (r.dst << 16) | (r.nf << 12) | (r.k << 8) | fl; };
    auto close_group = [&]() { if (gopen) { FgGroupHdr g; std::memcpy(&g, &P.d_chunks[ghdr], sizeof(g)); g.nrec = (uint16_t)gn; std::memcpy(&P.d_chunks[ghdr], &g, sizeof(g)); gopen = false; } };
    auto close_chunk = [&]() {
      close_group();
      if (!open) return;
      FgChunkHdr h; std::memset(&h, 0, sizeof(h)); h.ngroups = ngroups; std::memcpy(&P.d_chunks[base], &h, sizeof(h)); open = false;
      P.d_chunk_used.push_back((uint32_t)((cur + 15) & ~(size_t)15));
      // sequences of tensor-core groups of one class: length and byte size, stored in the first header of each run
      std::vector<size_t> offs, sizes; size_t o = base + sizeof(FgChunkHdr);
      for (int gi = 0; gi < ngroups; ++gi) {
        FgGroupHdr g; std::memcpy(&g, &P.d_chunks[o], sizeof(g));
        const bool qx = (g.flags & FG_REC_QEXT) != 0;
        size_t body = (g.flags & FG_REC_MMA) ? (size_t)g.nrec * (size_t)FG_TILE_BYTES(mma_steps(g.k, qx))
                                             : (size_t)g.nrec * (((g.flags & FG_REC_WIDE) ? sizeof(FgRecW) : sizeof(FgRecC)) + (size_t)rec_ncoef_host(g.k, g.flags) * sizeof(double));
        if (g.flags & FG_REC_MMA) { g.grp_units = (uint16_t)(body / 16); std::memcpy(&P.d_chunks[o], &g, sizeof(g)); }
        offs.push_back(o); sizes.push_back(sizeof(FgGroupHdr) + body); o += sizeof(FgGroupHdr) + body;
      }
      for (int gi = 0; gi < ngroups; ++gi) {
        FgGroupHdr g; std::memcpy(&g, &P.d_chunks[offs[gi]], sizeof(g));
        if (!(g.flags & FG_REC_MMA)) continue;
        int n = 1; size_t bytes = sizes[gi];
        for (int gj = gi + 1; gj < ngroups; ++gj) { FgGroupHdr g2; std::memcpy(&g2, &P.d_chunks[offs[gj]], sizeof(g2)); if (g2.nf != g.nf || g2.k != g.k || g2.flags != g.flags || g2.dst != g.dst) break; ++n; bytes += sizes[gj]; }
        g.nseq = (uint16_t)n; g.seq_units = (uint16_t)(bytes / 16); std::memcpy(&P.d_chunks[offs[gi]], &g, sizeof(g));
      }
    };
    auto new_chunk = [&]() { close_chunk(); base = P.d_chunks.size(); P.d_chunks.resize(base + FG_CHUNK_BYTES, 0); cur = sizeof(FgChunkHdr); ngroups = 0; open = true; };
    auto open_group = [&](const HRecord& r, int extra_flags) {
      close_group();
      FgGroupHdr g; std::memset(&g, 0, sizeof(g)); g.nf = (uint8_t)r.nf; g.k = (uint8_t)r.k; g.dst = (uint8_t)r.dst;
      g.flags = (uint8_t)((r.flags & (FG_REC_TWO | FG_REC_QEXT)) | (r.nf > FG_NFC ? FG_REC_WIDE : 0) | extra_flags);
      std::memcpy(g.vidx, r.vidx, sizeof(g.vidx));
      ghdr = base + cur; std::memcpy(&P.d_chunks[ghdr], &g, sizeof(g)); cur += sizeof(g); gopen = true; gn = 0; ++ngroups; prev = nullptr;
    };
    auto mma_coef = [](const HRecord& r, int step, int x, bool par4 = false) -> double {      // par4: the parity-homogeneous step order of flagged k = 4 groups
      const int k = r.k; const double* mainT = r.coef.data(); const double* qT = mainT + (1 << k); const int qs = (1 << k) >> 1;
      if (k < 2) return x == 0 ? mainT[0] : (x == 1 && k == 1) ? mainT[1] : (x == 2 && k == 1 && (r.flags & FG_REC_QEXT)) ? qT[0] : 0.0;      // {1, a0, aq0, 0}
      if (k == 4 && par4) {      // parity-homogeneous steps (fg_tables.h)
        if (step < 4) return mainT[FG_MMA4_MAIN_SUBSET(step, x)];
        const int j = (step - 4) >> 1, par = (step - 4) & 1; return qT[j * qs + FG_MMA4_Q_SUBSET(par, x)];
      }
      const int nm = 1 << (k - 2);
      if (step < nm) return mainT[x | (step << 2)];
      if (step < 2 * nm) { int t = step - nm, j = x >> 1; return qT[j * qs + ((x & 1) | (t << 1))]; }
      int s2 = step - 2 * nm, nh = (1 << k) >> 3, j = 2 + s2 / nh, t2 = s2 % nh; return qT[j * qs + (x | (t2 << 2))];
    };
    size_t nr = N.recs.size();
    for (size_t i = 0; i < nr;) {
      size_t j = i + 1;
      while (j < nr && cls(N.recs[j]) == cls(N.recs[i]) && std::memcmp(N.recs[j].vidx, N.recs[i].vidx, sizeof(N.recs[i].vidx)) == 0) ++j;
      const HRecord& r0 = N.recs[i];
      const bool qx = (r0.flags & FG_REC_QEXT) != 0;
      bool mma = r0.nf <= FG_NFC && !(r0.flags & FG_REC_TWO) && r0.k >= FG_MMA_MINK && (j - i) >= FG_MMA_MINREC;
      if (mma) {     // tiles store the high word of the double: only if every coefficient of the run has a zero low word
        for (size_t t = i; t < j && mma; ++t) for (double c : N.recs[t].coef) { FgMmaCoef h; if (!fg_mma_coef_pack(c, &h)) { mma = false; break; } }
      }
      if (mma) {
        const int steps = mma_steps(r0.k, qx); const size_t tile_bytes = (size_t)FG_TILE_BYTES(steps);
        const int R = (int)(j - i), ntiles = (R + 7) / 8;
        // record shown to lane c (of every quad) in tile t, slot e: depth-first index c*2*ntiles + 2t + e
        auto rec_at = [&](int t, int n) -> const HRecord* { int d = (n >> 1) * 2 * ntiles + 2 * t + (n & 1); return d < R ? &N.recs[i + d] : nullptr; };
        // k = 4: steps in which a record of the run has a non-zero coefficient; inside set A or set B the group is flagged
        // and the kernel leaves the other steps out
        int par_flag = 0, steps_run = steps;
        if (r0.k == 4 && FG_MMA_PARITY) {
          uint32_t gm = 0;
          for (size_t t = i; t < j; ++t) for (int st = 0; st < steps; ++st) for (int x = 0; x < 4; ++x) if (mma_coef(N.recs[t], st, x, true) != 0.0) gm |= 1u << st;
          if ((gm & ~FG_MMA_PAR_MASK_A(qx)) == 0) { par_flag = FG_REC_PAR_A; steps_run = __builtin_popcount(FG_MMA_PAR_MASK_A(qx)); }
          else if ((gm & ~FG_MMA_PAR_MASK_B(qx)) == 0) { par_flag = FG_REC_PAR_B; steps_run = __builtin_popcount(FG_MMA_PAR_MASK_B(qx)); }
        }
        for (int t = 0; t < ntiles; ++t) {
          bool need_group = !gopen || prev != nullptr;      // prev != nullptr: a regular group is open
          if (!open || cur + tile_bytes + (need_group ? sizeof(FgGroupHdr) : 0) > FG_CHUNK_BYTES) { new_chunk(); need_group = true; }
          if (need_group) open_group(r0, FG_REC_MMA | par_flag);
          for (int n = 0; n < 8; ++n) {
            FgRecM h; std::memset(&h, 0, sizeof(h)); h.keep = (uint8_t)r0.nf;
            if (const HRecord* r = rec_at(t, n)) {
              std::memcpy(h.fidx, r->fidx, FG_NFC); h.cab16 = fg_cab16_pack((double)std::max(r->cabs[0], r->cabs[1]));
              const HRecord* pr = (n & 1) ? rec_at(t, n - 1) : (t > 0 && gn > 0 ? rec_at(t - 1, n + 1) : nullptr);   // gn == 0: first tile of a (re)opened group
              int keep = 0; if (pr) while (keep < r->nf && r->fidx[keep] == pr->fidx[keep]) ++keep;
              h.keep = (uint8_t)keep;
              N.exec_flops += std::max(0, r->nf - std::max(keep, 1));
            }
            std::memcpy(&P.d_chunks[base + cur + n * sizeof(FgRecM)], &h, sizeof(h));
          }
          FgMmaCoef* fr = (FgMmaCoef*)&P.d_chunks[base + cur + 8 * sizeof(FgRecM)];
          for (int st = 0; st < steps; ++st) for (int n = 0; n < 8; ++n) for (int x = 0; x < 4; ++x) {
            const HRecord* r = rec_at(t, n); FgMmaCoef h = 0; if (r) fg_mma_coef_pack(mma_coef(*r, st, x, par_flag != 0), &h); fr[st * 32 + n * 4 + x] = h;
          }
          cur += tile_bytes; ++gn;
          N.exec_flops += 8.0 * (8.0 * steps_run + 4.0);
        }
        { auto& h = hist[{1, r0.nf, r0.k, qx ? 1 : 0, 0}]; h[0] += R; h[1] += ntiles; h[2] += 1; }
        if (std::getenv("FG_PLAN_HIST")) {      // sparsity by k-step: per record the mask of steps with a non-zero coefficient
          static std::map<std::vector<int>, std::map<unsigned, long>> masks; static std::map<std::vector<int>, std::array<long, 3>> tot;
          std::vector<int> key = {r0.nf, r0.k, qx ? 1 : 0};
          std::map<unsigned, long> local;
          for (size_t t = i; t < j; ++t) { unsigned m = 0; for (int st = 0; st < steps; ++st) for (int x = 0; x < 4; ++x) if (mma_coef(N.recs[t], st, x) != 0.0) m |= 1u << st; masks[key][m]++; local[m]++; tot[key][0] += __builtin_popcount(m); tot[key][1] += steps; }
          // tiles needed if the records of this run are regrouped by mask: sum over masks of ceil(count/8) * popcount(mask)
          long dm = 0; for (auto& kv : local) dm += ((kv.second + 7) / 8) * __builtin_popcount(kv.first);
          tot[key][2] += dm;
          if (i + R >= nr) for (auto& kv : tot) std::fprintf(stderr, "  steps nf %d k %d qx %d: nonzero record-steps %ld of %ld; DMMA per row block if regrouped by mask %ld; distinct masks %zu\n", kv.first[0], kv.first[1], kv.first[2], kv.second[0], kv.second[1], kv.second[2], masks[kv.first].size());
        }
        for (size_t t = i; t < j; ++t) N.algo_flops += std::max(0, N.recs[t].nf - 1);
        close_group();
        i = j; continue;
      }
      for (size_t t = i; t < j; ++t) {
        const HRecord& r = N.recs[t];
        const bool wide = r.nf > FG_NFC;
        size_t need = (wide ? sizeof(FgRecW) : sizeof(FgRecC)) + r.coef.size() * sizeof(double);
        bool newgroup = !gopen || !prev || cls(*prev) != cls(r) || gn >= 65535;
        if (!open || cur + need + (newgroup ? sizeof(FgGroupHdr) : 0) > FG_CHUNK_BYTES) { new_chunk(); newgroup = true; }
        if (newgroup) open_group(r, 0);
        int keep = 0;
        if (prev) while (keep < r.nf && keep < prev->nf && r.fidx[keep] == prev->fidx[keep]) ++keep;
        const float cab = std::max(r.cabs[0], r.cabs[1]);
        if (wide) { FgRecW h; std::memset(&h, 0, sizeof(h)); h.keep = (uint8_t)keep; std::memcpy(h.fidx, r.fidx, sizeof(h.fidx)); std::memcpy(h.vidx, r.vidx, sizeof(h.vidx)); h.cabs = cab; std::memcpy(&P.d_chunks[base + cur], &h, sizeof(h)); cur += sizeof(h); }
        else { FgRecC h; std::memset(&h, 0, sizeof(h)); h.keep = (uint8_t)keep; std::memcpy(h.fidx, r.fidx, sizeof(h.fidx)); std::memcpy(h.vidx, r.vidx, sizeof(h.vidx)); h.cabs = cab; std::memcpy(&P.d_chunks[base + cur], &h, sizeof(h)); cur += sizeof(h); }
        std::memcpy(&P.d_chunks[base + cur], r.coef.data(), r.coef.size() * sizeof(double)); cur += r.coef.size() * sizeof(double);
        ++gn; prev = &r;
        { auto& h = hist[{0, r.nf, r.k, (r.flags & FG_REC_QEXT) ? 1 : 0, (r.flags & FG_REC_TWO) ? 1 : 0}]; h[0] += 1; if (t == i) h[2] += 1; }
        const int nco = (r.flags & FG_REC_TWO) ? 2 : 1;
        N.exec_flops += std::max(0, r.nf - std::max(keep, 1)) + nco * (2.0 * ((1 << r.k) - 1) + 4.0) + ((r.flags & FG_REC_QEXT) ? r.k * (2.0 * ((1 << r.k) / 2 - 1) + 2.0) : 0.0);
        N.algo_flops += std::max(0, r.nf - std::max(keep, 1));
      }
      i = j;
    }
    close_chunk();
    d.chunk_count = (int)(P.d_chunks.size() / FG_CHUNK_BYTES) - d.chunk_begin;
    P.d_nums.push_back(d);
    P.d_geom_num_begin[N.geom + 1] = (int)i + 1;
    raw_max = std::max(raw_max, (1 << N.nse) * FG_NDEG * N.ncomp);
    P.n_records += (long)N.recs.size(); P.n_coefs += N.n_coefs; P.n_nonzero += N.n_nonzero;
    P.exec_flops += N.exec_flops; P.algo_flops += N.algo_flops;
    std::vector<HRecord>().swap(N.recs);   // the stream is the product; drop the host copy
  }
  for (size_t gi = 1; gi <= P.geoms.size(); ++gi) if (P.d_geom_num_begin[gi] < P.d_geom_num_begin[gi - 1]) P.d_geom_num_begin[gi] = P.d_geom_num_begin[gi - 1];
  for (auto& nd : P.nodes) {
    FgNodeDev d; std::memset(&d, 0, sizeof(d)); d.num = nd.num; d.ncomp = P.nums[nd.num].ncomp; d.nse = (int)nd.se_kid.size(); d.nvc = (int)nd.vc_kid.size();
    for (int k = 0; k < d.nse; ++k) d.se_kid[k] = nd.se_kid[k];
    for (int k = 0; k < d.nvc; ++k) d.vc_kid[k] = nd.vc_kid[k];
    P.d_nodes.push_back(d);
  }
  for (auto& t : P.terms) {
    FgTermDev d; std::memset(&d, 0, sizeof(d)); d.top = t.top; d.sign = t.sign; d.nmem = (int)t.geoms.size();
    for (int k = 0; k < d.nmem; ++k) d.geom[k] = t.geoms[k];
    P.d_terms.push_back(d);
  }
  if (std::getenv("FG_PLAN_HIST")) {
    std::fprintf(stderr, "fg_plan: record classes (mma nf k qx two): records tiles runs\n");
    for (auto& kv : hist) std::fprintf(stderr, "  %d %d %d %d %d : %ld %ld %ld\n", kv.first[0], kv.first[1], kv.first[2], kv.first[3], kv.first[4], kv.second[0], kv.second[1], kv.second[2]);
  }
  P.raw_slots = raw_max;
  // scratch per sample: [U,W per geom][raw value][raw abs][node value 2*NDEG][node abs 2*NDEG]
  P.scratch_slots = 2 * (int)P.geoms.size() + 2 * raw_max + 4 * FG_NDEG * (int)P.nodes.size();
  build_density(P);
  // algorithmic flops outside the numerator stream (rough, per sample): geometry + node products + assembly + sampler
  double extra = 0;
  for (auto& E : P.geoms) extra += 2.0 * (E.l * E.l * E.l / 3.0 + E.ne * E.l * E.l + E.ne * (E.ne + 1) / 2.0 * E.l + 4.0 * E.ne * E.l);
  extra += (double)P.nodes.size() * 2.0 * FG_NDEG * FG_NDEG + (double)P.terms.size() * 4.0 * n + 60.0 * P.M;
  P.algo_flops += extra; P.exec_flops += extra;
  P.plan_seconds = std::chrono::duration<double>(std::chrono::steady_clock::now() - t0).count();
  return FG_OK;
}

}  // namespace fg
