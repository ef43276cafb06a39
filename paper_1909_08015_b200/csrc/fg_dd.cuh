// fg_dd.cuh — double-double arithmetic (106-bit significand) for the first rung of the precision ladder
// (samples whose double-precision value is not trusted are recomputed at higher precision).
// Error-free transformations (Knuth two-sum, FMA two-product); no code shared with the CPU oracle.
#pragma once
#include <math.h>

#if defined(__CUDACC__)
#define FG_HD __host__ __device__ __forceinline__
#else
#define FG_HD inline
#endif

namespace fg {

#if defined(__CUDA_ARCH__)
FG_HD double f_add(double a, double b) { return __dadd_rn(a, b); }   // never contracted into an FMA
FG_HD double f_mul(double a, double b) { return __dmul_rn(a, b); }
FG_HD double f_fma(double a, double b, double c) { return __fma_rn(a, b, c); }
#else
FG_HD double f_add(double a, double b) { volatile double r = a + b; return r; }
FG_HD double f_mul(double a, double b) { volatile double r = a * b; return r; }
FG_HD double f_fma(double a, double b, double c) { return fma(a, b, c); }
#endif

struct dd {
  double hi, lo;
  FG_HD dd() : hi(0.0), lo(0.0) {}
  FG_HD dd(double h) : hi(h), lo(0.0) {}
  FG_HD dd(double h, double l) : hi(h), lo(l) {}
};

FG_HD dd two_sum(double a, double b) { double s = f_add(a, b), bb = f_add(s, -a); return dd(s, f_add(f_add(a, -f_add(s, -bb)), f_add(b, -bb))); }
FG_HD dd quick_two_sum(double a, double b) { double s = f_add(a, b); return dd(s, f_add(b, -f_add(s, -a))); }
FG_HD dd two_prod(double a, double b) { double p = f_mul(a, b); return dd(p, f_fma(a, b, -p)); }

FG_HD dd operator+(dd a, dd b) {      // "sloppy" sum: error <= 2^-104 (|a| + |b|); cancellation is accounted for by the |.| sums
  dd s = two_sum(a.hi, b.hi);
  s.lo = f_add(s.lo, f_add(a.lo, b.lo));
  return quick_two_sum(s.hi, s.lo);
}
FG_HD dd operator-(dd a) { return dd(-a.hi, -a.lo); }
FG_HD dd operator-(dd a, dd b) { return a + (-b); }
FG_HD dd operator*(dd a, dd b) {
  dd p = two_prod(a.hi, b.hi);
  p.lo = f_add(p.lo, f_add(f_mul(a.hi, b.lo), f_mul(a.lo, b.hi)));
  return quick_two_sum(p.hi, p.lo);
}
FG_HD dd operator*(dd a, double b) { dd p = two_prod(a.hi, b); p.lo = f_fma(a.lo, b, p.lo); return quick_two_sum(p.hi, p.lo); }
FG_HD dd operator/(dd a, dd b) {
  double q1 = a.hi / b.hi; dd r = a - b * q1;
  double q2 = r.hi / b.hi; r = r - b * q2;
  double q3 = r.hi / b.hi;
  dd q = quick_two_sum(q1, q2); return q + dd(q3);
}
FG_HD dd dd_add_d(dd a, double b) { dd s = two_sum(a.hi, b); s.lo = f_add(s.lo, a.lo); return quick_two_sum(s.hi, s.lo); }

// generic helpers used by the evaluator templates (T = double or dd)
FG_HD double to_double(double a) { return a; }
FG_HD double to_double(dd a) { return a.hi + a.lo; }
FG_HD double t_abs_d(double a) { return fabs(a); }
FG_HD double t_abs_d(dd a) { return fabs(a.hi); }
FG_HD double t_fma(double a, double b, double c) { return fma(a, b, c); }
FG_HD dd t_fma(dd a, dd b, dd c) { return a * b + c; }
FG_HD double t_halve(double a) { return 0.5 * a; }
FG_HD dd t_halve(dd a) { return dd(0.5 * a.hi, 0.5 * a.lo); }
template <class T> struct is_dd { static const bool value = false; };
template <> struct is_dd<dd> { static const bool value = true; };

}  // namespace fg
