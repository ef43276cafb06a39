// fg_core.cuh — per-sample arithmetic of the hot path, written once for T = double and T = dd.
//   a1 Philox4x32-10 stream
//   a2-a4 Hepp-sector sample, coordinates, pdf
//   a5 element geometry: loop matrix, LDL^T, U, W, A, A^q, beta   PAPER.md:205 (method by reference)
//   a6 numerator stream interpreter
//   a7 forest sum
// Everything here is device code; the FG_HD qualifier only lets a developer harness instantiate the same
// templates on the host for debugging.  The library itself has no CPU compute path.
#pragma once
#include <float.h>
#include <stdint.h>

#include "fg_dd.cuh"
#include "fg_qd.cuh"
#include "fg_tables.h"

namespace fg {

// ------------------------------------------------------------------------------------------------
// a1  Philox4x32-10: counter = (sample_lo, sample_hi, call, 0), key = (seed_lo, seed_hi)
// ------------------------------------------------------------------------------------------------
FG_HD void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0, uint32_t k1, uint32_t out[4]) {
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    uint64_t p0 = (uint64_t)0xD2511F53u * c0, p1 = (uint64_t)0xCD9E8D57u * c2;
    uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0, n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
    c1 = (uint32_t)p1; c3 = (uint32_t)p0; c0 = n0; c2 = n2;
    k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}
// 53-bit uniform in the open interval (0,1)
FG_HD double uniform53(uint32_t w0, uint32_t w1) { return ((double)((((uint64_t)w0 << 32) | w1) >> 11) + 0.5) * 0x1p-53; }

// Second stream: MRG32k3a (L'Ecuyer 1999): x1_n = (1403580 x1_{n-2} - 810728 x1_{n-3}) mod (2^32 - 209),
// x2_n = (527612 x2_{n-1} - 1370589 x2_{n-3}) mod (2^32 - 22853), u = ((x1 - x2) mod m1) / (m1 + 1) in (0, 1).  Sample `sid`
// owns outputs 32 sid, 32 sid + 1, ...: its state is reached from the seed's with the precomputed powers A^(32 2^j) of the
// two recurrence matrices, one matrix-vector product mod m per set bit of sid (fg.h, option rng).
#define FG_MRG_M1 4294967087ull
#define FG_MRG_M2 4294944443ull
struct UniformStream {
  uint64_t sid, seed; uint32_t call, w[4]; int left; int rng; uint32_t s1[3], s2[3];
  FG_HD UniformStream(uint64_t sid_, uint64_t seed_, int rng_ = 0, const uint32_t* __restrict__ jump = nullptr) : sid(sid_), seed(seed_), call(0), left(0), rng(rng_) {
    if (rng == 1) {
      for (int i = 0; i < 3; ++i) { s1[i] = (uint32_t)(1ull + ((seed & 0xffffffffull) * (uint64_t)(i + 1) + 12344ull) % (FG_MRG_M1 - 1ull)); s2[i] = (uint32_t)(1ull + ((seed >> 32) * (uint64_t)(i + 1) + 12344ull) % (FG_MRG_M2 - 1ull)); }
      for (int j = 0; j < FG_MRG_JUMPS && (sid >> j) != 0; ++j) if ((sid >> j) & 1ull) {
        const uint32_t* A = jump + 18 * j; uint32_t r1[3], r2[3];
        for (int i = 0; i < 3; ++i) {      // three products below 2^64 / 3 each: reduce every product, then the sum
          r1[i] = (uint32_t)(((uint64_t)A[3 * i] * s1[0] % FG_MRG_M1 + (uint64_t)A[3 * i + 1] * s1[1] % FG_MRG_M1 + (uint64_t)A[3 * i + 2] * s1[2] % FG_MRG_M1) % FG_MRG_M1);
          r2[i] = (uint32_t)(((uint64_t)A[9 + 3 * i] * s2[0] % FG_MRG_M2 + (uint64_t)A[9 + 3 * i + 1] * s2[1] % FG_MRG_M2 + (uint64_t)A[9 + 3 * i + 2] * s2[2] % FG_MRG_M2) % FG_MRG_M2);
        }
        for (int i = 0; i < 3; ++i) { s1[i] = r1[i]; s2[i] = r2[i]; }
      }
    }
  }
  FG_HD double next_mrg() {
    const uint64_t p1 = (1403580ull * s1[1] + 810728ull * (FG_MRG_M1 - s1[0])) % FG_MRG_M1;
    const uint64_t p2 = (527612ull * s2[2] + 1370589ull * (FG_MRG_M2 - s2[0])) % FG_MRG_M2;
    s1[0] = s1[1]; s1[1] = s1[2]; s1[2] = (uint32_t)p1; s2[0] = s2[1]; s2[1] = s2[2]; s2[2] = (uint32_t)p2;
    return (double)(p1 > p2 ? p1 - p2 : p1 + FG_MRG_M1 - p2) * 2.328306549295727688e-10;
  }
  FG_HD double next() {
    if (rng == 1) return next_mrg();
    if (left == 0) { philox4x32_10((uint32_t)sid, (uint32_t)(sid >> 32), call++, 0u, (uint32_t)seed, (uint32_t)(seed >> 32), w); left = 2; }
    double u = (left == 2) ? uniform53(w[0], w[1]) : uniform53(w[2], w[3]);
    --left; return u;
  }
};

// ------------------------------------------------------------------------------------------------
// a2-a4  one sample of g = sum_k C_k g_k.  g_k has the form (14) with exponent table Deg_k:
//   k=0: Deg_1 (graph table, through Z_1);  k=1: Deg = 1/2;  k=2: D*Deg_1 (through Z_3);  k=3: Deg(s) = |s| (uniform).
// Sector j_1..j_M is drawn by M categorical draws with weights Z(s \ j); tau_l = u^(1/Deg(s_l)); z_{j_l} ~ prod tau.
// The selection sums are evaluated in ascending line order without FMA contraction (bit-exact sectors).
// ------------------------------------------------------------------------------------------------
struct Sample { double z[FG_MAXM]; uint8_t order[FG_MAXM]; double mant; int ex; int comp; bool bad; };

FG_HD void draw_sample(const FgPlanDev& P, const double* __restrict__ Z1, const double* __restrict__ Z3, uint64_t sid, uint64_t seed, Sample& r) {
  const int M = P.M; const uint32_t full = (1u << M) - 1u;
  UniformStream us(sid, seed, P.rng, P.mrg_jump);
  double uc = us.next();
  int comp = 3; { double c = 0.0; for (int k = 0; k < 4; ++k) { c = f_add(c, P.C[k]); if (uc < c) { comp = k; break; } } }
  r.comp = comp;
  double zeta[FG_MAXM], lnr[FG_MAXM], d1[FG_MAXM];
  uint32_t s = full; double zprev = 1.0;
  for (int l = 0; l < M; ++l) {
    const int cnt = __builtin_popcount(s);
    double tot1 = 0.0;
    for (int j = 0; j < M; ++j) if ((s >> j) & 1u) tot1 = f_add(tot1, Z1[s ^ (1u << j)]);
    d1[l] = (l == 0) ? 0.0 : tot1 / Z1[s];          // Deg_1(s) = sum_j Z_1(s\j) / Z_1(s)
    const double usel = us.next();
    int pick = -1;
    if (comp == 0 || comp == 2) {
      const double* Z = (comp == 0) ? Z1 : Z3;
      double tot = tot1;
      if (comp == 2) { tot = 0.0; for (int j = 0; j < M; ++j) if ((s >> j) & 1u) tot = f_add(tot, Z[s ^ (1u << j)]); }
      const double thr = f_mul(usel, tot); double cum = 0.0; int last = -1;
      for (int j = 0; j < M; ++j) if ((s >> j) & 1u) { cum = f_add(cum, Z[s ^ (1u << j)]); last = j; if (cum > thr) { pick = j; break; } }
      if (pick < 0) pick = last;
    } else {
      int k = (int)f_mul(usel, (double)cnt); if (k >= cnt) k = cnt - 1;
      for (int j = 0; j < M; ++j) if ((s >> j) & 1u) { if (k == 0) { pick = j; break; } --k; }
    }
    if (l == 0) { zeta[0] = 1.0; lnr[0] = 0.0; }
    else {
      const double dg = (comp == 0) ? d1[l] : (comp == 1) ? 0.5 : (comp == 2) ? f_mul(P.D, d1[l]) : (double)cnt;
      const double u = us.next();
      lnr[l] = log(u) / dg;                          // ln(z_{j_l} / z_{j_{l-1}})
      zeta[l] = f_mul(zprev, pow(u, 1.0 / dg));
    }
    zprev = zeta[l];
    r.order[l] = (uint8_t)pick; s ^= (1u << pick);
  }
  double sum = 0.0; for (int l = 0; l < M; ++l) sum = f_add(sum, zeta[l]);
  bool bad = false;
  for (int l = 0; l < M; ++l) { double zz = zeta[l] / sum; r.z[r.order[l]] = zz; if (!(zz >= DBL_MIN)) bad = true; }
  // ln g_k = -ln Z_k(full) + sum_{l>=2} Deg_k(s_l) ln(z_{j_l}/z_{j_{l-1}}) - sum_j ln z_j      (14)
  double lnzeta = 0.0, lnz_sum = 0.0;
  for (int l = 0; l < M; ++l) { lnzeta += lnr[l]; lnz_sum += lnzeta; }
  lnz_sum -= M * log(sum);
  double lg[4];
  for (int k = 0; k < 4; ++k) {
    double e = 0.0;
    for (int l = 1; l < M; ++l) { double dk = (k == 0) ? d1[l] : (k == 1) ? 0.5 : (k == 2) ? f_mul(P.D, d1[l]) : (double)(M - l); e += dk * lnr[l]; }
    lg[k] = -P.lnZfull[k] + e - lnz_sum;
  }
  double mx = -DBL_MAX; for (int k = 0; k < 4; ++k) if (P.C[k] > 0.0 && lg[k] > mx) mx = lg[k];
  double acc = 0.0; for (int k = 0; k < 4; ++k) if (P.C[k] > 0.0) acc += P.C[k] * exp(lg[k] - mx);
  // g = acc * e^mx kept as mant * 2^ex with mant in [0.5,1)
  const double l2 = mx * 1.4426950408889634074, fl = floor(l2);
  int e2; const double mant = frexp(acc * exp2(l2 - fl), &e2);
  r.mant = mant; r.ex = e2 + (int)fl;
  if (!(mant > 0.0) || !(mant < 1.0)) bad = true;
  r.bad = bad;
}

// ------------------------------------------------------------------------------------------------
// a5  geometry of one element at one point.  Loop a = own photon a plus the own electron lines between its ends:
//   B_ab = sum_j z_j eta_ja eta_jb + delta_ab z_gamma_a,  U = det B,  C_a = sum_j z_j eta_ja,  W = C^T B^-1 C,
//   A_j = 1 - eta_j^T B^-1 C,  beta_ij = eta_i^T B^-1 eta_j,  A^q_j = xi^q_j - eta_j^T B^-1 C^q.
// B = L D L^T (no square roots).  This step is carried out in double-double for the double and the double-double rung
// (quad-double for the quad-double rung), whatever the precision of the numerator pass: it is a few per cent of the work at 5 loops and it removes the cancellations of the pivots,
// of 1 - sum and of the beta dot products from the double-precision pass.
// V receives beta (upper triangle, row-major), then A, then A^q, element idx at V[idx * vs]; amax = max(1,|A|,|A^q|);
// amp = conditioning of this step: product of the pivot ratios B_aa/d_a times the worst ratio sum|terms|/|value| of the
// final sums of A, A^q and beta (relative error of the entries of V is about amp * 2^-104).
// ------------------------------------------------------------------------------------------------
// G = arithmetic of the geometry step: double-double for the double and double-double rungs, quad-double for the last one
template <class T> struct geom_prec { typedef dd type; };
template <> struct geom_prec<qd> { typedef qd type; };
template <class T, class G> FG_HD T from_geom(const G& a);
template <> FG_HD double from_geom<double, dd>(const dd& a) { return a.hi + a.lo; }
template <> FG_HD dd from_geom<dd, dd>(const dd& a) { return a; }
template <> FG_HD qd from_geom<qd, qd>(const qd& a) { return a; }
FG_HD double g_hi(const dd& a) { return a.hi; }
FG_HD double g_hi(const qd& a) { return a.x[0]; }
FG_HD dd g_add_d(const dd& a, double b) { return dd_add_d(a, b); }
FG_HD qd g_add_d(const qd& a, double b) { return a + qd(b); }

template <class T>
FG_HD void geom_eval(const FgGeomDev& E, const double* zl, T* V, int vs, T& U, T& W, double& amax, double& amp) {
  typedef typename geom_prec<T>::type G;
  const int l = E.l, ne = E.ne;
  G B[FG_MAXL][FG_MAXL], C[FG_MAXL], Cq[FG_MAXL], invd[FG_MAXL];
  for (int a = 0; a < l; ++a) { C[a] = G(0.0); Cq[a] = G(0.0); for (int b = 0; b < l; ++b) B[a][b] = G(0.0); }
  for (int q = 0; q < ne; ++q) {
    const double z = zl[E.line_e[q]]; const unsigned m = E.eta[q]; const int xq = E.xiq[q];
    const double zh = xq > 0 ? 0.5 * z : -0.5 * z;
    for (int a = 0; a < l; ++a) if ((m >> a) & 1u) {
      C[a] = g_add_d(C[a], z);
      if (xq != 0) Cq[a] = g_add_d(Cq[a], zh);
      for (int b = 0; b <= a; ++b) if ((m >> b) & 1u) B[a][b] = g_add_d(B[a][b], z);
    }
  }
  for (int a = 0; a < l; ++a) B[a][a] = g_add_d(B[a][a], zl[E.line_ph[a]]);
  G u(1.0); double growth = 1.0;
  for (int a = 0; a < l; ++a) {
    G d = B[a][a]; const double baa = g_hi(d);
    for (int b = 0; b < a; ++b) d = d - B[a][b] * B[a][b] * B[b][b];     // B[b][b] holds d_b, B[a][b] holds L_ab
    invd[a] = G(1.0) / d; u = u * d; growth *= fmax(1.0, baa / g_hi(d));
    for (int c = a + 1; c < l; ++c) {
      G t = B[c][a];
      for (int b = 0; b < a; ++b) t = t - B[c][b] * B[a][b] * B[b][b];
      B[c][a] = t * invd[a];
    }
    B[a][a] = d;
  }
  U = from_geom<T, G>(u);
  for (int a = 0; a < l; ++a) for (int b = 0; b < a; ++b) { C[a] = C[a] - B[a][b] * C[b]; Cq[a] = Cq[a] - B[a][b] * Cq[b]; }   // L^-1 C, L^-1 C^q
  G w(0.0); for (int a = 0; a < l; ++a) { w = w + C[a] * C[a] * invd[a]; C[a] = C[a] * invd[a]; Cq[a] = Cq[a] * invd[a]; }
  W = from_geom<T, G>(w);
  G Y[FG_MAXNE][FG_MAXL]; int first[FG_MAXNE];
  const int nb = ne * (ne + 1) / 2; double am = 1.0, cond = 1.0;
  for (int q = 0; q < ne; ++q) {
    const unsigned m = E.eta[q];
    // y = L^-1 eta_q vanishes below the first loop of the line: structural zeros (block-uniform) are skipped everywhere
    int fq = 0; while (fq < l && !((m >> fq) & 1u)) ++fq;
    first[q] = fq;
    for (int a = 0; a < fq; ++a) Y[q][a] = G(0.0);
    for (int a = fq; a < l; ++a) { G y = ((m >> a) & 1u) ? G(1.0) : G(0.0); for (int b = fq; b < a; ++b) y = y - B[a][b] * Y[q][b]; Y[q][a] = y; }
    G sa(0.0), sq(0.0); double ta = 1.0, tq = 0.5;
    for (int a = fq; a < l; ++a) { const G t1 = Y[q][a] * C[a], t2 = Y[q][a] * Cq[a]; sa = sa + t1; sq = sq + t2; ta += fabs(g_hi(t1)); tq += fabs(g_hi(t2)); }
    const G A = G(1.0) - sa, Aq = G(0.5 * (double)E.xiq[q]) - sq;
    V[(nb + q) * vs] = from_geom<T, G>(A); V[(nb + ne + q) * vs] = from_geom<T, G>(Aq);
    am = fmax(am, fmax(fabs(g_hi(A)), fabs(g_hi(Aq))));
    if (g_hi(A) != 0.0) cond = fmax(cond, ta / fabs(g_hi(A)));
    if (E.xiq[q] != 0 && g_hi(Aq) != 0.0) cond = fmax(cond, tq / fabs(g_hi(Aq)));
  }
  amax = am;
  int idx = 0;
  for (int i = 0; i < ne; ++i) {
    G yd[FG_MAXL]; for (int a = first[i]; a < l; ++a) yd[a] = Y[i][a] * invd[a];
    for (int j = i; j < ne; ++j) {
      const int f2 = first[i] > first[j] ? first[i] : first[j];
      G b(0.0); double tb = 0.0; for (int a = f2; a < l; ++a) { const G t1 = yd[a] * Y[j][a]; b = b + t1; tb += fabs(g_hi(t1)); }
      if (g_hi(b) != 0.0) cond = fmax(cond, tb / fabs(g_hi(b)));
      V[idx * vs] = from_geom<T, G>(b); ++idx;
    }
  }
  amp = growth * cond;
}

// ------------------------------------------------------------------------------------------------
// a6  multilinear polynomial in K variables with a dense 2^K coefficient table (uniform across the block)
// ------------------------------------------------------------------------------------------------
template <class T, int S, int K, bool AC = false, bool RC = false> struct Horner {   // AC: use |coef|; RC: coefs already in registers
  static FG_HD void run(const double* __restrict__ c, const T (*a)[S], T* out) {
    T lo[S], hi[S];
    Horner<T, S, K - 1, AC, RC>::run(c, a, lo); Horner<T, S, K - 1, AC, RC>::run(c + (1 << (K - 1)), a, hi);
#pragma unroll
    for (int s = 0; s < S; ++s) out[s] = t_fma(a[K - 1][s], hi[s], lo[s]);
  }
};
template <class T, int S, bool AC, bool RC> struct Horner<T, S, 0, AC, RC> {
  static FG_HD void run(const double* __restrict__ c, const T (*)[S], T* out) {
    const double c0 = AC ? fabs(c[0]) : c[0];
#pragma unroll
    for (int s = 0; s < S; ++s) out[s] = T(c0);
  }
};
#if defined(__CUDACC__)
FG_HD void ld_coef2(const double* __restrict__ c, double& c0, double& c1) { const double2 v = *reinterpret_cast<const double2*>(c); c0 = v.x; c1 = v.y; }   // one 128-bit (broadcast) load
#else
FG_HD void ld_coef2(const double* __restrict__ c, double& c0, double& c1) { c0 = c[0]; c1 = c[1]; }
#endif
template <int S, bool AC, bool RC> struct Horner<double, S, 1, AC, RC> {   // leaf FMA takes both coefficients straight from the table (16-byte aligned)
  static FG_HD void run(const double* __restrict__ c, const double (*a)[S], double* out) {
    double c0, c1;
    if (RC) { c0 = c[0]; c1 = c[1]; } else ld_coef2(c, c0, c1);
    if (AC) { c0 = fabs(c0); c1 = fabs(c1); }
#pragma unroll
    for (int s = 0; s < S; ++s) out[s] = fma(a[0][s], c1, c0);
  }
};
// q-extension: q += sum_j aq[j] * (multilinear in the K-1 variables other than j)
template <class T, int S, int K, bool AC = false, bool RC = false> struct QExt {
  static FG_HD void run(const double* __restrict__ cq, const T (*a)[S], const T (*aq)[S], T* q) {
#pragma unroll
    for (int j = 0; j < K; ++j) {
      T b[K > 1 ? K - 1 : 1][S], sub[S];
#pragma unroll
      for (int i = 0; i + 1 < K; ++i) {
#pragma unroll
        for (int s = 0; s < S; ++s) b[i][s] = a[i < j ? i : i + 1][s];
      }
      Horner<T, S, K - 1, AC, RC>::run(cq + j * (1 << (K - 1)), b, sub);
#pragma unroll
      for (int s = 0; s < S; ++s) q[s] = t_fma(aq[j][s], sub[s], q[s]);
    }
  }
};
template <class T, int S, bool AC, bool RC> struct QExt<T, S, 0, AC, RC> { static FG_HD void run(const double*, const T (*)[S], const T (*)[S], T*) {} };

// Running state of one program: accumulators of the current destination.  split = w (0 = off, else 2..32): groups of w adjacent lanes evaluate the SAME point
// and share its records out (record i goes to lane i % w); their partial sums are added when a destination is finished
// (short double-double queues).
template <class T, int S> struct RecState { T acc[2][S]; double aab[2][S]; int cur, split, rr;
#ifdef FG_PHASE_PROF
  long long* prof; long long tlast;
#endif
};
// Phase cycle counters of a profiling build (-DFG_PHASE_PROF; fg_plan_phase_cycles): per warp, clock64 deltas between marks.
// 0 sampler, 1 geometry, 2 tensor-core groups, 3 static scalar groups, 4 dynamic groups, 5 ring wait + chunk barrier,
// 6 node products, 7 forest sum + weights + tail, 8 program set-up / flush
#if defined(FG_PHASE_PROF) && defined(__CUDA_ARCH__)
#define FG_MARK(obj, i) do { const long long t_ = clock64(); (obj).prof[i] += t_ - (obj).tlast; (obj).tlast = t_; } while (0)
#else
#define FG_MARK(obj, i) do { } while (0)
#endif

FG_HD constexpr int rec_ncoef(int k, int flags) {
  return (((flags & FG_REC_QEXT) ? (1 << k) + k * ((1 << k) >> 1) : ((flags & FG_REC_TWO) ? 2 : 1) << k) + 1) & ~1;
}

#if defined(__CUDACC__)
template <int I, int N> struct PreLoad {
  static __device__ __forceinline__ void run(unsigned caddr, double* cr) {
    asm volatile("ld.shared.v2.f64 {%0, %1}, [%2+%3];" : "=d"(cr[I]), "=d"(cr[I + 1]) : "r"(caddr), "n"(I * 8));
    PreLoad<I + 2, N>::run(caddr, cr);
  }
};
template <int N> struct PreLoad<N, N> { static __device__ __forceinline__ void run(unsigned, double*) {} };
#endif

// One group of compact records, class known at compile time: the inner loop has no data-dependent control flow
// except the (block-uniform) prefix depth `keep`.  Kept out of line on the device so that every class gets its own
// register allocation and instruction schedule (the accumulators travel through memory once per group).
// The coefficients of a record are read into registers first (128-bit broadcast loads, all in flight together),
// then consumed by the FMA tree: the shared-memory latency is paid once per record, not once per FMA.
#if defined(__CUDACC__)
#define FG_NOINLINE __device__ __noinline__
#else
#define FG_NOINLINE inline
#endif
#if defined(__CUDACC__)
#define FG_FORCEINLINE __device__ __forceinline__
#else
#define FG_FORCEINLINE inline
#endif
template <class T, int S, int ABS, int NF, int K, bool QX>
FG_FORCEINLINE void run_group_static_body(const unsigned char* __restrict__ p, int nrec, const T* __restrict__ Vt, int vs, int ne, T* __restrict__ accp, double* __restrict__ aabp, int r0 = 0) {   // records r0 .. nrec-1 (r0 > 0: a second thread set takes the rest; its first record rebuilds the whole prefix)
#if defined(__CUDA_ARCH__)
  __builtin_assume(__isShared(p)); __builtin_assume(__isShared(Vt));
#endif
  constexpr int FL = QX ? FG_REC_QEXT : 0;
  constexpr int NC = rec_ncoef(K, FL);
  constexpr int STRIDE = (int)sizeof(FgRecC) + NC * (int)sizeof(double);
  constexpr bool PRELOAD = NC <= 48;      // tables small enough to sit in registers
  T pf[NF > 0 ? NF : 1][S], acc[S]; double aab[S];
  T a[K > 0 ? K : 1][S], aq[K > 0 ? K : 1][S]; uint32_t lastv = 0xffffffffu;
#pragma unroll
  for (int s = 0; s < S; ++s) { acc[s] = accp[s]; aab[s] = aabp[s]; }
  p += (size_t)r0 * STRIDE;
  for (int r = r0; r < nrec; ++r, p += STRIDE) {
    const FgRecC h = *(const FgRecC*)p;
    const double* __restrict__ coef = (const double*)(p + sizeof(FgRecC));
    double cr[PRELOAD ? NC : 2];
    if (PRELOAD) {
#if defined(__CUDA_ARCH__)
      // volatile PTX keeps these loads together at the head of the record (the compiler otherwise sinks each load
      // next to its FMA and the warp pays the shared-memory latency once per FMA pair)
      const unsigned caddr = (unsigned)__cvta_generic_to_shared(coef);
      PreLoad<0, NC>::run(caddr, cr);
#else
      for (int i = 0; i < NC; ++i) cr[i] = coef[i];
#endif
    }
    const double* __restrict__ cc = PRELOAD ? cr : coef;
    const int keep = (r == r0 && r0 > 0) ? 0 : h.keep;
    // levels keep .. NF-1 of the prefix stack are rebuilt.  keep is the same in every lane (all lanes run the same record):
    // a uniform switch with fall-through, so that every level is defined unconditionally inside its case
    switch (keep) {
#define FG_LVL(F) case F: if (F < NF) { const T* pv = Vt + (int)h.fidx[F < NF ? F : 0] * vs; _Pragma("unroll") for (int s = 0; s < S; ++s) pf[F < NF ? F : 0][s] = (F == 0) ? pv[s] : pf[(F > 0 && F < NF) ? F - 1 : 0][s] * pv[s]; }
      FG_LVL(0) FG_LVL(1) FG_LVL(2) FG_LVL(3) FG_LVL(4) FG_LVL(5)
#undef FG_LVL
      default: break;
    }
    // free variables: reloaded only when they change (runs of records share them)
    uint32_t vkey; __builtin_memcpy(&vkey, h.vidx, 4);
    if (K > 0 && vkey != lastv) {
      lastv = vkey;
#pragma unroll
      for (int j = 0; j < K; ++j) {
        const T* pv = Vt + (int)h.vidx[j] * vs;
#pragma unroll
        for (int s = 0; s < S; ++s) a[j][s] = pv[s];
        if (QX) {
          const T* pq = pv + ne * vs;
#pragma unroll
          for (int s = 0; s < S; ++s) aq[j][s] = pq[s];
        }
      }
    }
#if defined(__CUDA_ARCH__) && defined(FG_STATIC_SYNCWARP)
    __syncwarp();   // scheduling fence: every load of the record is issued before the first FMA waits on one
#endif
    T q[S];
    Horner<T, S, K, false, PRELOAD>::run(cc, a, q);
    if (QX) QExt<T, S, K, false, PRELOAD>::run(cc + (1 << K), a, aq, q);
    const double cab = (double)h.cabs;
#pragma unroll
    for (int s = 0; s < S; ++s) {
      if (NF > 0) { acc[s] = t_fma(pf[NF > 0 ? NF - 1 : 0][s], q[s], acc[s]); if (ABS) aab[s] = fma(t_abs_d(pf[NF > 0 ? NF - 1 : 0][s]), cab, aab[s]); }
      else { acc[s] = acc[s] + q[s]; if (ABS) aab[s] += cab; }
    }
  }
#pragma unroll
  for (int s = 0; s < S; ++s) { accp[s] = acc[s]; aabp[s] = aab[s]; }
}

template <class T, int S, int ABS, int NF, int K, bool QX>
FG_NOINLINE void run_group_static(const unsigned char* __restrict__ p, int nrec, const T* __restrict__ Vt, int vs, int ne, T* __restrict__ accp, double* __restrict__ aabp, int r0 = 0) {
  run_group_static_body<T, S, ABS, NF, K, QX>(p, nrec, Vt, vs, ne, accp, aabp, r0);
}

FG_HD int fg_lane() {
#if defined(__CUDA_ARCH__)
  return (int)(threadIdx.x & 31);
#else
  return 0;
#endif
}
#if defined(__CUDACC__)
__device__ __forceinline__ double warp_sum(double v, int w) { for (int o = w >> 1; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o); return v; }
__device__ __forceinline__ dd warp_sum(dd v, int w) { for (int o = w >> 1; o > 0; o >>= 1) v = v + dd(__shfl_xor_sync(0xffffffffu, v.hi, o), __shfl_xor_sync(0xffffffffu, v.lo, o)); return v; }
__device__ __forceinline__ qd warp_sum(qd v, int w) {
  for (int o = w >> 1; o > 0; o >>= 1) v = v + qd(__shfl_xor_sync(0xffffffffu, v.x[0], o), __shfl_xor_sync(0xffffffffu, v.x[1], o), __shfl_xor_sync(0xffffffffu, v.x[2], o), __shfl_xor_sync(0xffffffffu, v.x[3], o));
  return v;
}
#endif
// split mode (st.split = w = 2..32 lanes per point): add the partial sums of the w lanes of a point (each of them ends up
// with the same totals)
template <class T, int S>
FG_HD void fold_split(RecState<T, S>& st) {
#if defined(__CUDA_ARCH__)
  if (st.split) {
#pragma unroll
    for (int c = 0; c < 2; ++c) {
#pragma unroll
      for (int s = 0; s < S; ++s) { st.acc[c][s] = warp_sum(st.acc[c][s], st.split); st.aab[c][s] = warp_sum(st.aab[c][s], st.split); }
    }
  }
#endif
}

// One group of any class, everything dynamic (wide records, two-component records, the double-double pass).
template <class T, int S, int ABS>
FG_HD void run_group_dyn(const unsigned char* __restrict__ p, int nrec, int nf, int k, int flags, const T* __restrict__ Vt, int vs, int ne, RecState<T, S>& st) {
  const bool wide = (flags & FG_REC_WIDE) != 0;
  const int stride = (wide ? (int)sizeof(FgRecW) : (int)sizeof(FgRecC)) + rec_ncoef(k, flags) * (int)sizeof(double);
  // split mode: record i of the running count goes to lane i % w of the point; every lane walks its own records
  int r0 = 0, rstep = 1;
  if (st.split) { r0 = (fg_lane() - st.rr) & (st.split - 1); rstep = st.split; st.rr += nrec; }
  p += (size_t)r0 * stride;
  for (int r = r0; r < nrec; r += rstep, p += (size_t)rstep * stride) {
    const uint8_t* fidx = wide ? ((const FgRecW*)p)->fidx : ((const FgRecC*)p)->fidx;
    const uint8_t* vidx = wide ? ((const FgRecW*)p)->vidx : ((const FgRecC*)p)->vidx;
    const double cab = wide ? (double)((const FgRecW*)p)->cabs : (double)((const FgRecC*)p)->cabs;
    const double* __restrict__ coef = (const double*)(p + (wide ? sizeof(FgRecW) : sizeof(FgRecC)));
    T prod[S];
#pragma unroll
    for (int s = 0; s < S; ++s) prod[s] = T(1.0);
    for (int f = 0; f < nf; ++f) {
      const T* pv = Vt + (int)fidx[f] * vs;
#pragma unroll
      for (int s = 0; s < S; ++s) prod[s] = prod[s] * pv[s];
    }
    T a[FG_KMAX][S], aq[FG_KMAX][S];
#pragma unroll
    for (int j = 0; j < FG_KMAX; ++j) if (j < k) {
      const T* pv = Vt + (int)vidx[j] * vs;
#pragma unroll
      for (int s = 0; s < S; ++s) { a[j][s] = pv[s]; aq[j][s] = (flags & FG_REC_QEXT) ? pv[ne * vs + s] : T(0.0); }
    }
    T q[2][S]; double qa[2][S];
    switch (k) {
#define FG_CASE(K) case K: Horner<T, S, K>::run(coef, a, q[0]); \
                           if (flags & FG_REC_TWO) Horner<T, S, K>::run(coef + (1 << K), a, q[1]); \
                           else if (flags & FG_REC_QEXT) QExt<T, S, K>::run(coef + (1 << K), a, aq, q[0]); break;
      FG_CASE(0) FG_CASE(1) FG_CASE(2) FG_CASE(3) FG_CASE(4)
#undef FG_CASE
      default: break;
    }
    if (ABS == 2) {
      double ab[FG_KMAX][S], abq[FG_KMAX][S];
#pragma unroll
      for (int j = 0; j < FG_KMAX; ++j) if (j < k) {
#pragma unroll
        for (int s = 0; s < S; ++s) { ab[j][s] = t_abs_d(a[j][s]); abq[j][s] = t_abs_d(aq[j][s]); }
      }
      switch (k) {
#define FG_CASE(K) case K: Horner<double, S, K, true>::run(coef, ab, qa[0]); \
                           if (flags & FG_REC_TWO) Horner<double, S, K, true>::run(coef + (1 << K), ab, qa[1]); \
                           else if (flags & FG_REC_QEXT) QExt<double, S, K, true>::run(coef + (1 << K), ab, abq, qa[0]); break;
        FG_CASE(0) FG_CASE(1) FG_CASE(2) FG_CASE(3) FG_CASE(4)
#undef FG_CASE
        default: break;
      }
    }
#pragma unroll
    for (int s = 0; s < S; ++s) {
      st.acc[0][s] = t_fma(prod[s], q[0][s], st.acc[0][s]);
      if (ABS == 1) st.aab[0][s] = fma(t_abs_d(prod[s]), cab, st.aab[0][s]);
      if (ABS == 2) st.aab[0][s] = fma(t_abs_d(prod[s]), qa[0][s], st.aab[0][s]);
      if (flags & FG_REC_TWO) {
        st.acc[1][s] = t_fma(prod[s], q[1][s], st.acc[1][s]);
        if (ABS == 1) st.aab[1][s] = fma(t_abs_d(prod[s]), cab, st.aab[1][s]);
        if (ABS == 2) st.aab[1][s] = fma(t_abs_d(prod[s]), qa[1][s], st.aab[1][s]);
      }
    }
  }
}

// ---- tensor-core groups (FG_REC_MMA): monomial order shared by the planner, the scalar interpreter and the DMMA path ----
FG_HD constexpr int mma_steps(int k, bool qx) { return k < 2 ? 1 : (1 << (k - 2)) + (qx ? (1 << (k - 2)) + (k - 2) * ((1 << k) >> 3) : 0); }

// all monomials of one point: mono[4*step + x] (see FgRecM in fg_tables.h)
template <class T>
FG_HD void mma_monomials(int k, bool qx, bool par4, const T* a, const T* aq, T* mono) {      // par4: group flagged FG_REC_PAR_A / FG_REC_PAR_B
  if (k < 2) { mono[0] = T(1.0); mono[1] = k ? a[0] : T(0.0); mono[2] = (k && qx) ? aq[0] : T(0.0); mono[3] = T(0.0); return; }
  const int nm = 1 << (k - 2);
  if (k == 4 && par4) {      // parity-homogeneous steps (fg_tables.h): subsets of the four variables, of the other three
    for (int st = 0; st < 4; ++st) for (int x = 0; x < 4; ++x) {
      const int sub = FG_MMA4_MAIN_SUBSET(st, x); T m = T(1.0);
      for (int i = 0; i < 4; ++i) if ((sub >> i) & 1) m = m * a[i];
      mono[4 * st + x] = m;
    }
    if (qx) for (int j = 0; j < 4; ++j) for (int par = 0; par < 2; ++par) for (int x = 0; x < 4; ++x) {
      const int sub = FG_MMA4_Q_SUBSET(par, x); T m = aq[j]; int bit = 0;
      for (int i = 0; i < 4; ++i) if (i != j) { if ((sub >> bit) & 1) m = m * a[i]; ++bit; }
      mono[4 * (4 + 2 * j + par) + x] = m;
    }
    return;
  }
  T mlo[4] = {T(1.0), a[0], a[1], a[0] * a[1]};
  for (int t = 0; t < nm; ++t) {
    T h = T(1.0); for (int i = 0; i + 2 < k; ++i) if ((t >> i) & 1) h = h * a[2 + i];
    for (int x = 0; x < 4; ++x) mono[4 * t + x] = mlo[x] * h;
    if (qx) {
      mono[4 * (nm + t) + 0] = aq[0] * h; mono[4 * (nm + t) + 1] = aq[0] * a[1] * h;
      mono[4 * (nm + t) + 2] = aq[1] * h; mono[4 * (nm + t) + 3] = aq[1] * a[0] * h;
    }
  }
  if (qx) {
    const int nh = (1 << k) >> 3; int step = 2 * nm;
    for (int j = 2; j < k; ++j) for (int t2 = 0; t2 < nh; ++t2, ++step) {
      T h = aq[j]; int bit = 0;
      for (int i = 2; i < k; ++i) if (i != j) { if ((t2 >> bit) & 1) h = h * a[i]; ++bit; }
      for (int x = 0; x < 4; ++x) mono[4 * step + x] = mlo[x] * h;
    }
  }
}

// scalar interpreter of a tensor-core group (double-double pass, host harness): one point per thread
template <class T, int S, int ABS>
FG_HD void run_group_mma_dyn(const unsigned char* __restrict__ p, int ntiles, int nf, int k, int flags, const uint8_t* vidx, const T* __restrict__ Vt, int vs, int ne, RecState<T, S>& st) {
  const bool qx = (flags & FG_REC_QEXT) != 0; const int steps = mma_steps(k, qx);
  T mono[S][48]; double monoa[S][48];
#pragma unroll
  for (int s = 0; s < S; ++s) {
    T a[FG_KMAX], aq[FG_KMAX];
    for (int j = 0; j < k; ++j) { a[j] = Vt[(int)vidx[j] * vs + s]; aq[j] = qx ? Vt[((int)vidx[j] + ne) * vs + s] : T(0.0); }
    mma_monomials<T>(k, qx, (flags & (FG_REC_PAR_A | FG_REC_PAR_B)) != 0, a, aq, mono[s]);
    if (ABS == 2) for (int J = 0; J < 4 * steps; ++J) monoa[s][J] = t_abs_d(mono[s][J]);
  }
  const int tile_bytes = FG_TILE_BYTES(steps);
  int q0 = 0, qstep = 1;
  if (st.split) { q0 = (fg_lane() - st.rr) & (st.split - 1); qstep = st.split; st.rr += ntiles * 8; }
  for (int q = q0; q < ntiles * 8; q += qstep) {
    const int t = q >> 3, n = q & 7;
    const unsigned char* pt = p + (size_t)t * tile_bytes;
    const FgRecM* recs = (const FgRecM*)pt; const FgMmaCoef* __restrict__ fr = (const FgMmaCoef*)(pt + 8 * sizeof(FgRecM));
    const double cab = fg_cab16_value(recs[n].cab16);
#pragma unroll
    for (int s = 0; s < S; ++s) {
      T qv = T(0.0); double qa = 0.0;
      for (int J = 0; J < 4 * steps; ++J) { const double c = fg_mma_coef_value(fr[(J >> 2) * 32 + n * 4 + (J & 3)]); qv = qv + mono[s][J] * T(c); if (ABS == 2) qa += monoa[s][J] * fabs(c); }
      T bp = T(1.0); for (int f = 0; f < nf; ++f) bp = bp * Vt[(int)recs[n].fidx[f] * vs + s];
      st.acc[0][s] = st.acc[0][s] + bp * qv;
      if (ABS == 1) st.aab[0][s] = fma(t_abs_d(bp), cab, st.aab[0][s]);
      if (ABS == 2) st.aab[0][s] = fma(t_abs_d(bp), qa, st.aab[0][s]);
    }
  }
}

// All groups of one chunk.  flush(dst, acc, aab) stores the finished accumulators of a destination.
// ABS: 0 no |.| tracking, 1 bound by cabs (needs |A|,|A^q| <= 1), 2 exact sum of |coef| prod |A| in double
template <class T, int S, int ABS, class Flush>
FG_HD void run_chunk(const unsigned char* __restrict__ chunk, const T* __restrict__ Vt, int vs, int ne, RecState<T, S>& st, Flush&& flush) {
#if defined(__CUDA_ARCH__)
  __builtin_assume(__isShared(chunk)); __builtin_assume(__isShared(Vt));   // LDS instead of generic loads
#endif
  const int ngroups = ((const FgChunkHdr*)chunk)->ngroups;
  const unsigned char* p = chunk + sizeof(FgChunkHdr);
  for (int g = 0; g < ngroups; ++g) {
    FG_MARK(st, 8);
    const FgGroupHdr gh = *(const FgGroupHdr*)p; p += sizeof(FgGroupHdr);
    const int nrec = gh.nrec, nf = gh.nf, k = gh.k, flags = gh.flags;
    if ((int)gh.dst != st.cur) {
      if (st.cur >= 0) { fold_split(st); flush(st.cur, st.acc, st.aab); }
      st.cur = gh.dst;
#pragma unroll
      for (int s = 0; s < S; ++s) { st.acc[0][s] = T(0.0); st.acc[1][s] = T(0.0); st.aab[0][s] = 0.0; st.aab[1][s] = 0.0; }
    }
    bool done = false;
    if constexpr (!is_ext<T>::value && ABS != 2) {      // (host harness; the device's double pass has its own chunk loop, fg_stream.cuh)
      if (!(flags & (FG_REC_WIDE | FG_REC_TWO | FG_REC_MMA))) {
        done = true;
        const bool qx = (flags & FG_REC_QEXT) != 0;
        switch (nf * 8 + k) {
#define FG_CLS(NF, K) case NF * 8 + K: if (qx) run_group_static<T, S, ABS, NF, K, true>(p, nrec, Vt, vs, ne, st.acc[0], st.aab[0]); \
                                        else run_group_static<T, S, ABS, NF, K, false>(p, nrec, Vt, vs, ne, st.acc[0], st.aab[0]); break;
          FG_CLS(0, 0) FG_CLS(0, 1) FG_CLS(0, 2) FG_CLS(0, 3) FG_CLS(0, 4)
          FG_CLS(1, 0) FG_CLS(1, 1) FG_CLS(1, 2) FG_CLS(1, 3) FG_CLS(1, 4)
          FG_CLS(2, 0) FG_CLS(2, 1) FG_CLS(2, 2) FG_CLS(2, 3) FG_CLS(2, 4)
          FG_CLS(3, 0) FG_CLS(3, 1) FG_CLS(3, 2) FG_CLS(3, 3) FG_CLS(3, 4)
          FG_CLS(4, 0) FG_CLS(4, 1) FG_CLS(4, 2) FG_CLS(4, 3) FG_CLS(4, 4)
          FG_CLS(5, 0) FG_CLS(5, 1) FG_CLS(5, 2) FG_CLS(5, 3) FG_CLS(5, 4)
#undef FG_CLS
          default: done = false; break;
        }
      }
    }
    if (flags & FG_REC_MMA) {
      if (!done) run_group_mma_dyn<T, S, ABS>(p, nrec, nf, k, flags, gh.vidx, Vt, vs, ne, st);
      FG_MARK(st, 4);
      p += (size_t)gh.grp_units * 16;
      continue;
    }
    if (!done) { run_group_dyn<T, S, ABS>(p, nrec, nf, k, flags, Vt, vs, ne, st); FG_MARK(st, 4); } else FG_MARK(st, 3);
    p += nrec * (((flags & FG_REC_WIDE) ? (int)sizeof(FgRecW) : (int)sizeof(FgRecC)) + rec_ncoef(k, flags) * (int)sizeof(double));
  }
}

// Scratch layout per sample (slot index; element at Sc[slot * ss]):
//   [0, 2*ngeom)                U_g, W_g
//   [rawv, rawv + raw_slots)    raw accumulators R[sig][deg][comp] of the running program; then their |.| sums
//   node value polynomials [node][comp][deg], then node |.| polynomials
struct ScratchMap {
  int rawv, rawa, nodev, nodea;
  FG_HD ScratchMap(const FgPlanDev& P) { rawv = 2 * P.ngeom; rawa = rawv + P.raw_slots; nodev = rawa + P.raw_slots; nodea = nodev + 2 * FG_NDEG * P.nnode; }
};

// a6 (cont.)  After the stream of a program: node polynomial = sum_sig R[sig] * prod_i (u or v of self-energy kid i),
// times the scalar polynomials of the vertexlike kids.  Polynomials in t, degree < FG_NDEG.
template <class T, bool ABS>
FG_HD void finish_node(const FgPlanDev& P, const ScratchMap& sm, int node_id, T* Sc, int ss) {
  const FgNodeDev nd = P.nodes[node_id];
  const int nc = nd.ncomp, raw0 = ABS ? sm.rawa : sm.rawv, node0 = ABS ? sm.nodea : sm.nodev;
  T out[2][FG_NDEG];
  for (int c = 0; c < 2; ++c) for (int d = 0; d < FG_NDEG; ++d) out[c][d] = T(0.0);
  for (int sig = 0; sig < (1 << nd.nse); ++sig) {
    T f[FG_NDEG]; f[0] = T(1.0); for (int d = 1; d < FG_NDEG; ++d) f[d] = T(0.0);
    for (int i = 0; i < nd.nse; ++i) {
      const T* kp = Sc + (node0 + (nd.se_kid[i] * 2 + ((sig >> i) & 1)) * FG_NDEG) * ss;
      T g[FG_NDEG]; for (int d = 0; d < FG_NDEG; ++d) g[d] = T(0.0);
      for (int d1 = 0; d1 < FG_NDEG; ++d1) for (int d2 = 0; d1 + d2 < FG_NDEG; ++d2) g[d1 + d2] = g[d1 + d2] + f[d1] * kp[d2 * ss];
      for (int d = 0; d < FG_NDEG; ++d) f[d] = g[d];
    }
    for (int c = 0; c < nc; ++c) for (int d1 = 0; d1 < FG_NDEG; ++d1) {
      const T r = Sc[(raw0 + (sig * FG_NDEG + d1) * nc + c) * ss];
      for (int d2 = 0; d1 + d2 < FG_NDEG; ++d2) out[c][d1 + d2] = out[c][d1 + d2] + r * f[d2];
    }
  }
  for (int i = 0; i < nd.nvc; ++i) {
    const T* kp = Sc + (node0 + (nd.vc_kid[i] * 2) * FG_NDEG) * ss;
    for (int c = 0; c < nc; ++c) {
      T g[FG_NDEG]; for (int d = 0; d < FG_NDEG; ++d) g[d] = T(0.0);
      for (int d1 = 0; d1 < FG_NDEG; ++d1) for (int d2 = 0; d1 + d2 < FG_NDEG; ++d2) g[d1 + d2] = g[d1 + d2] + out[c][d1] * kp[d2 * ss];
      for (int d = 0; d < FG_NDEG; ++d) out[c][d] = g[d];
    }
  }
  for (int c = 0; c < nc; ++c) for (int d = 0; d < FG_NDEG; ++d) Sc[(node0 + (node_id * 2 + c) * FG_NDEG + d) * ss] = out[c][d];
}

// a7  I(z) = sum_{(F,G')} (-1)^{|F|-1} prod_S[(-1/4)^{l_S} / U_S^2] sum_{m<n} (n-m-1)! P_m / W_F^{n-m}
template <class T, bool ABS>
FG_HD void assemble(const FgPlanDev& P, const ScratchMap& sm, const T* Sc, int ss, T& I, T& Iabs) {
  const int n = P.n;
  T tot = T(0.0), tota = T(0.0);
  for (int t = 0; t < P.nterm; ++t) {
    const FgTermDev tm = P.terms[t];
    T pu = T(1.0), wf = T(0.0);
    for (int k = 0; k < tm.nmem; ++k) { const T u = Sc[(2 * tm.geom[k]) * ss]; pu = pu * u * u; wf = wf + Sc[(2 * tm.geom[k] + 1) * ss]; }
    const T winv = T(1.0) / wf; T wp = winv, s = T(0.0), sa = T(0.0);
    const T* pv = Sc + (sm.nodev + tm.top * 2 * FG_NDEG) * ss; const T* pa = Sc + (sm.nodea + tm.top * 2 * FG_NDEG) * ss;
    for (int m = n - 1; m >= 0; --m) {
      const T fw = wp * T(P.fact[n - m - 1]);
      s = s + fw * pv[m * ss];
      if (ABS) sa = sa + fw * pa[m * ss];
      wp = wp * winv;
    }
    const T ipu = T(P.quarter_pow) / pu;
    const T val = s * ipu;
    tot = (tm.sign > 0) ? tot + val : tot - val;
    if (ABS) { const T va = sa * ipu; tota = tota + T(t_abs_d(va)); }
  }
  I = tot; Iabs = tota;
}

}  // namespace fg
