// fg_qd.cuh — quad-double arithmetic (four doubles, ~209-bit significand) for the last rung of the precision ladder
// (the paper goes double IA -> 128 -> 192 -> 256-bit mantissa; here double -> double-double ->
// quad-double).  Unevaluated sums of four doubles with the renormalisation-based algorithms of Hida, Li and Bailey
// ("Algorithms for quad-double precision floating point arithmetic", 2001), restated here with the error-free
// transformations of fg_dd.cuh.  The "sloppy" variants are used: relative error of one operation <= ~2^-205.
// Only the queued (ill-conditioned) samples ever reach this type, so the operators are kept out of line.
#pragma once
#include "fg_dd.cuh"

#if defined(__CUDACC__)
#define FG_QD_FN __host__ __device__ __noinline__
#else
#define FG_QD_FN inline
#endif

namespace fg {

struct qd {
  double x[4];
  FG_HD qd() { x[0] = x[1] = x[2] = x[3] = 0.0; }
  FG_HD qd(double a) { x[0] = a; x[1] = x[2] = x[3] = 0.0; }
  FG_HD qd(dd a) { x[0] = a.hi; x[1] = a.lo; x[2] = x[3] = 0.0; }
  FG_HD qd(double a, double b, double c, double d) { x[0] = a; x[1] = b; x[2] = c; x[3] = d; }
};

FG_HD void qd_two_sum(double a, double b, double& s, double& e) { const dd t = two_sum(a, b); s = t.hi; e = t.lo; }
FG_HD void qd_quick_two_sum(double a, double b, double& s, double& e) { const dd t = quick_two_sum(a, b); s = t.hi; e = t.lo; }
FG_HD void qd_two_prod(double a, double b, double& p, double& e) { const dd t = two_prod(a, b); p = t.hi; e = t.lo; }
FG_HD void qd_three_sum(double& a, double& b, double& c) {
  double t1, t2, t3; qd_two_sum(a, b, t1, t2); qd_two_sum(c, t1, a, t3); qd_two_sum(t2, t3, b, c);
}
FG_HD void qd_three_sum2(double& a, double& b, double c) {
  double t1, t2, t3; qd_two_sum(a, b, t1, t2); qd_two_sum(c, t1, a, t3); b = f_add(t2, t3);
}

// five overlapping components -> four non-overlapping ones
FG_HD qd qd_renorm(double c0, double c1, double c2, double c3, double c4) {
  double s0, s1, s2 = 0.0, s3 = 0.0;
  qd_quick_two_sum(c3, c4, s0, c4); qd_quick_two_sum(c2, s0, s0, c3); qd_quick_two_sum(c1, s0, s0, c2); qd_quick_two_sum(c0, s0, c0, c1);
  s0 = c0; s1 = c1;
  if (s1 != 0.0) {
    qd_quick_two_sum(s1, c2, s1, s2);
    if (s2 != 0.0) { qd_quick_two_sum(s2, c3, s2, s3); if (s3 != 0.0) s3 = f_add(s3, c4); else qd_quick_two_sum(s2, c4, s2, s3); }
    else { qd_quick_two_sum(s1, c3, s1, s2); if (s2 != 0.0) qd_quick_two_sum(s2, c4, s2, s3); else qd_quick_two_sum(s1, c4, s1, s2); }
  } else {
    qd_quick_two_sum(s0, c2, s0, s1);
    if (s1 != 0.0) { qd_quick_two_sum(s1, c3, s1, s2); if (s2 != 0.0) qd_quick_two_sum(s2, c4, s2, s3); else qd_quick_two_sum(s1, c4, s1, s2); }
    else { qd_quick_two_sum(s0, c3, s0, s1); if (s1 != 0.0) qd_quick_two_sum(s1, c4, s1, s2); else qd_quick_two_sum(s0, c4, s0, s1); }
  }
  return qd(s0, s1, s2, s3);
}

FG_QD_FN qd qd_add(const qd& a, const qd& b) {
  double s0, s1, s2, s3, t0, t1, t2, t3;
  qd_two_sum(a.x[0], b.x[0], s0, t0); qd_two_sum(a.x[1], b.x[1], s1, t1); qd_two_sum(a.x[2], b.x[2], s2, t2); qd_two_sum(a.x[3], b.x[3], s3, t3);
  qd_two_sum(s1, t0, s1, t0);
  qd_three_sum(s2, t0, t1);
  qd_three_sum2(s3, t0, t2);
  t0 = f_add(f_add(t0, t1), t3);
  return qd_renorm(s0, s1, s2, s3, t0);
}

FG_QD_FN qd qd_mul(const qd& a, const qd& b) {
  double p0, p1, p2, p3, p4, p5, q0, q1, q2, q3, q4, q5, t0, t1, s0, s1, s2;
  qd_two_prod(a.x[0], b.x[0], p0, q0);
  qd_two_prod(a.x[0], b.x[1], p1, q1); qd_two_prod(a.x[1], b.x[0], p2, q2);
  qd_two_prod(a.x[0], b.x[2], p3, q3); qd_two_prod(a.x[1], b.x[1], p4, q4); qd_two_prod(a.x[2], b.x[0], p5, q5);
  qd_three_sum(p1, p2, q0);                       // start the accumulation
  qd_three_sum(p2, q1, q2); qd_three_sum(p3, p4, p5);   // six three-sums for p2, q1, q2, p3, p4, p5
  qd_two_sum(p2, p3, s0, t0); qd_two_sum(q1, p4, s1, t1);
  s2 = f_add(q2, p5);
  qd_two_sum(s1, t0, s1, t0);
  s2 = f_add(s2, f_add(t0, t1));
  // O(eps^3) terms
  s1 = f_add(s1, f_add(f_add(f_add(f_mul(a.x[0], b.x[3]), f_mul(a.x[1], b.x[2])), f_add(f_mul(a.x[2], b.x[1]), f_mul(a.x[3], b.x[0]))), f_add(f_add(q0, q3), f_add(q4, q5))));
  return qd_renorm(p0, p1, s0, s1, s2);
}

FG_HD qd operator+(const qd& a, const qd& b) { return qd_add(a, b); }
FG_HD qd operator-(const qd& a) { return qd(-a.x[0], -a.x[1], -a.x[2], -a.x[3]); }
FG_HD qd operator-(const qd& a, const qd& b) { return qd_add(a, -b); }
FG_HD qd operator*(const qd& a, const qd& b) { return qd_mul(a, b); }
FG_QD_FN qd qd_div(const qd& a, const qd& b) {     // long division, five quotient digits
  double q0, q1, q2, q3, q4;
  q0 = a.x[0] / b.x[0]; qd r = a - b * qd(q0);
  q1 = r.x[0] / b.x[0]; r = r - b * qd(q1);
  q2 = r.x[0] / b.x[0]; r = r - b * qd(q2);
  q3 = r.x[0] / b.x[0]; r = r - b * qd(q3);
  q4 = r.x[0] / b.x[0];
  return qd_renorm(q0, q1, q2, q3, q4);
}
FG_HD qd operator/(const qd& a, const qd& b) { return qd_div(a, b); }

FG_HD double to_double(const qd& a) { return a.x[0] + a.x[1]; }
FG_HD double t_abs_d(const qd& a) { return fabs(a.x[0]); }
FG_HD qd t_fma(const qd& a, const qd& b, const qd& c) { return a * b + c; }
FG_HD qd t_halve(const qd& a) { return qd(0.5 * a.x[0], 0.5 * a.x[1], 0.5 * a.x[2], 0.5 * a.x[3]); }

// extended types (double-double, quad-double): the rungs that run the scalar interpreter with exact |.| sums
template <class T> struct is_ext { static const bool value = false; };
template <> struct is_ext<dd> { static const bool value = true; };
template <> struct is_ext<qd> { static const bool value = true; };

}  // namespace fg
