// ia_interval.cuh - device interval library (layer B0) for sm_100a.
//
// Intervals [lo, hi] with outward rounding from the hardware's directed-rounding instructions:
// DADD/DMUL/DFMA .RM/.RP (FADD/FMUL/FFMA .RM/.RP for the FP32 variant) issue at the same rate as
// their round-to-nearest forms, so an interval add is two FP64-pipe instructions and a
// sign-known interval multiply is two.  Arithmetic primitives return the tightest enclosure
// IEEE-754 allows; sin/cos/atan2 are CUDA's round-to-nearest routines (documented maximum error
// 2 ulp in double; sinf/cosf 2 ulp, atan2f 3 ulp in float) widened by a relative 2^-50 (2^-21 in
// float), i.e. between IA_PAD_ULPS = 4 and 8 ulps on each side, then clamped to the mathematical
// range.  The method these serve: the interval extension of eq. (4), PAPER.md L74-78 (ref [7]).
#pragma once
#include <cuda_runtime.h>
#include <math_constants.h>

#define IA_PAD_ULPS 4
#define IA_DEV __device__ __forceinline__

namespace ia {

template <class T> struct Iv { T lo, hi; };

// ---- directed scalar operations -------------------------------------------------------------
template <class T> struct Rnd;
template <> struct Rnd<double> {
  static IA_DEV double add_dn(double a, double b) { return __dadd_rd(a, b); }
  static IA_DEV double add_up(double a, double b) { return __dadd_ru(a, b); }
  static IA_DEV double mul_dn(double a, double b) { return __dmul_rd(a, b); }
  static IA_DEV double mul_up(double a, double b) { return __dmul_ru(a, b); }
  static IA_DEV double fma_dn(double a, double b, double c) { return __fma_rd(a, b, c); }
  static IA_DEV double fma_up(double a, double b, double c) { return __fma_ru(a, b, c); }
  static IA_DEV double div_dn(double a, double b) { return __ddiv_rd(a, b); }
  static IA_DEV double div_up(double a, double b) { return __ddiv_ru(a, b); }
  static IA_DEV double sqrt_dn(double a) { return __dsqrt_rd(a); }
  static IA_DEV double sqrt_up(double a) { return __dsqrt_ru(a); }
  static IA_DEV double add_rn(double a, double b) { return __dadd_rn(a, b); }   // never contracted
  static IA_DEV double mul_rn(double a, double b) { return __dmul_rn(a, b); }
  static IA_DEV double from_dn(double x) { return x; }
  static IA_DEV double from_up(double x) { return x; }
  static IA_DEV double from_rn(double x) { return x; }
  static IA_DEV double pad_rel() { return 0x1p-50; }
  static IA_DEV double pi_hi() { return 0x1.921fb54442d19p+1; }      // RU(pi)
  static IA_DEV double pi_lo() { return 0x1.921fb54442d18p+1; }      // RD(pi)
  static IA_DEV double pio2_hi() { return 0x1.921fb54442d19p+0; }
  static IA_DEV double pio2_lo() { return 0x1.921fb54442d18p+0; }
  static IA_DEV double el_sin(double x) { return sin(x); }
  static IA_DEV double el_cos(double x) { return cos(x); }
  static IA_DEV double el_atan2(double y, double x) { return atan2(y, x); }
};
template <> struct Rnd<float> {
  static IA_DEV float add_dn(float a, float b) { return __fadd_rd(a, b); }
  static IA_DEV float add_up(float a, float b) { return __fadd_ru(a, b); }
  static IA_DEV float mul_dn(float a, float b) { return __fmul_rd(a, b); }
  static IA_DEV float mul_up(float a, float b) { return __fmul_ru(a, b); }
  static IA_DEV float fma_dn(float a, float b, float c) { return __fmaf_rd(a, b, c); }
  static IA_DEV float fma_up(float a, float b, float c) { return __fmaf_ru(a, b, c); }
  static IA_DEV float div_dn(float a, float b) { return __fdiv_rd(a, b); }
  static IA_DEV float div_up(float a, float b) { return __fdiv_ru(a, b); }
  static IA_DEV float sqrt_dn(float a) { return __fsqrt_rd(a); }
  static IA_DEV float sqrt_up(float a) { return __fsqrt_ru(a); }
  static IA_DEV float add_rn(float a, float b) { return __fadd_rn(a, b); }
  static IA_DEV float mul_rn(float a, float b) { return __fmul_rn(a, b); }
  static IA_DEV float from_dn(double x) { return __double2float_rd(x); }
  static IA_DEV float from_up(double x) { return __double2float_ru(x); }
  static IA_DEV float from_rn(double x) { return __double2float_rn(x); }
  static IA_DEV float pad_rel() { return 0x1p-21f; }
  static IA_DEV float pi_hi() { return 0x1.921fb6p+1f; }
  static IA_DEV float pi_lo() { return 0x1.921fb4p+1f; }
  static IA_DEV float pio2_hi() { return 0x1.921fb6p+0f; }
  static IA_DEV float pio2_lo() { return 0x1.921fb4p+0f; }
  static IA_DEV float el_sin(float x) { return sinf(x); }
  static IA_DEV float el_cos(float x) { return cosf(x); }
  static IA_DEV float el_atan2(float y, float x) { return atan2f(y, x); }
};

// min/max as one compare + select (no NaN fix-up: NaN never wins the first slot twice; callers
// that care about NaN test the final enclosure with negated comparisons)
template <class T> IA_DEV T mn(T a, T b) { return a < b ? a : b; }
template <class T> IA_DEV T mx(T a, T b) { return a > b ? a : b; }

// ---- interval primitives --------------------------------------------------------------------
template <class T> IA_DEV Iv<T> thin(T x) { return {x, x}; }
template <class T> IA_DEV Iv<T> ineg(Iv<T> a) { return {-a.hi, -a.lo}; }
template <class T> IA_DEV Iv<T> iadd(Iv<T> a, Iv<T> b) { return {Rnd<T>::add_dn(a.lo, b.lo), Rnd<T>::add_up(a.hi, b.hi)}; }
template <class T> IA_DEV Iv<T> isub(Iv<T> a, Iv<T> b) { return {Rnd<T>::add_dn(a.lo, -b.hi), Rnd<T>::add_up(a.hi, -b.lo)}; }
template <class T> IA_DEV Iv<T> iadd_s(Iv<T> a, T c) { return {Rnd<T>::add_dn(a.lo, c), Rnd<T>::add_up(a.hi, c)}; }

// general product: min / max of the four endpoint products
template <class T> IA_DEV Iv<T> imul(Iv<T> a, Iv<T> b) {
  using R = Rnd<T>;
  T l = mn(mn(R::mul_dn(a.lo, b.lo), R::mul_dn(a.lo, b.hi)), mn(R::mul_dn(a.hi, b.lo), R::mul_dn(a.hi, b.hi)));
  T h = mx(mx(R::mul_up(a.lo, b.lo), R::mul_up(a.lo, b.hi)), mx(R::mul_up(a.hi, b.lo), R::mul_up(a.hi, b.hi)));
  return {l, h};
}
// a >= 0 (a.lo >= 0), b of any sign: the partner of each endpoint of b is chosen by its sign
template <class T> IA_DEV Iv<T> imul_pu(Iv<T> a, Iv<T> b) {
  using R = Rnd<T>;
  return {R::mul_dn(b.lo < T(0) ? a.hi : a.lo, b.lo), R::mul_up(b.hi < T(0) ? a.lo : a.hi, b.hi)};
}
// a >= 0 and b >= 0
template <class T> IA_DEV Iv<T> imul_pp(Iv<T> a, Iv<T> b) { return {Rnd<T>::mul_dn(a.lo, b.lo), Rnd<T>::mul_up(a.hi, b.hi)}; }
// exact scalar times interval
template <class T> IA_DEV Iv<T> iscale(T c, Iv<T> a) {
  using R = Rnd<T>;
  if (c >= T(0)) return {R::mul_dn(c, a.lo), R::mul_up(c, a.hi)};
  return {R::mul_dn(c, a.hi), R::mul_up(c, a.lo)};
}
template <class T> IA_DEV Iv<T> iscale_pos(T c, Iv<T> a) { return {Rnd<T>::mul_dn(c, a.lo), Rnd<T>::mul_up(c, a.hi)}; }
template <class T> IA_DEV Iv<T> isqr(Iv<T> a) {
  using R = Rnd<T>;
  if (a.lo >= T(0)) return {R::mul_dn(a.lo, a.lo), R::mul_up(a.hi, a.hi)};
  if (a.hi <= T(0)) return {R::mul_dn(a.hi, a.hi), R::mul_up(a.lo, a.lo)};
  return {T(0), mx(R::mul_up(a.lo, a.lo), R::mul_up(a.hi, a.hi))};
}
// branch-free form of the same: mig = smallest magnitude (0 if straddling), mag = largest
template <class T> IA_DEV Iv<T> isqr_bf(Iv<T> a) {
  using R = Rnd<T>;
  T mig = mx(mx(a.lo, -a.hi), T(0));
  T mag = mx(-a.lo, a.hi);
  return {R::mul_dn(mig, mig), R::mul_up(mag, mag)};
}
// a / b, b.lo > 0
template <class T> IA_DEV Iv<T> idiv_pos(Iv<T> a, Iv<T> b) {
  using R = Rnd<T>;
  T l = a.lo >= T(0) ? R::div_dn(a.lo, b.hi) : R::div_dn(a.lo, b.lo);
  T h = a.hi >= T(0) ? R::div_up(a.hi, b.lo) : R::div_up(a.hi, b.hi);
  return {l, h};
}
template <class T> IA_DEV Iv<T> irecip_pos(Iv<T> b) { return {Rnd<T>::div_dn(T(1), b.hi), Rnd<T>::div_up(T(1), b.lo)}; }
template <class T> IA_DEV Iv<T> isqrt(Iv<T> a) { return {Rnd<T>::sqrt_dn(mx(a.lo, T(0))), Rnd<T>::sqrt_up(mx(a.hi, T(0)))}; }
template <class T> IA_DEV Iv<T> iclamp(Iv<T> a, T lo, T hi) { return {mx(a.lo, lo), mn(a.hi, hi)}; }

// ---- elementary enclosures ------------------------------------------------------------------
// x -/+ |x| * 2^-50: between 4 and 8 ulps outward (the relative spacing of doubles is in
// (2^-53, 2^-52]); one directed FMA each
template <class T> IA_DEV T pad_dn(T x) { return Rnd<T>::fma_dn(-fabs(x), Rnd<T>::pad_rel(), x); }
template <class T> IA_DEV T pad_up(T x) { return Rnd<T>::fma_up(fabs(x), Rnd<T>::pad_rel(), x); }

// sin over e.  Outside [-4,4] (or NaN): [-1,1].  Inside, the interior critical points are
// +pi/2 (maximum) and -pi/2 (minimum) only.
template <class T> IA_DEV Iv<T> isin(Iv<T> e) {
  using R = Rnd<T>;
  if (!(e.lo >= T(-4) && e.hi <= T(4))) return {T(-1), T(1)};
  T a = R::el_sin(e.lo), b = R::el_sin(e.hi);
  Iv<T> r = {pad_dn(mn(a, b)), pad_up(mx(a, b))};
  if (e.lo <= R::pio2_hi() && e.hi >= R::pio2_lo()) r.hi = T(1);
  if (e.lo <= -R::pio2_lo() && e.hi >= -R::pio2_hi()) r.lo = T(-1);
  return iclamp(r, T(-1), T(1));
}
// cos over e: interior critical points inside [-4,4] are 0 (maximum) and +-pi (minimum).
template <class T> IA_DEV Iv<T> icos(Iv<T> e) {
  using R = Rnd<T>;
  if (!(e.lo >= T(-4) && e.hi <= T(4))) return {T(-1), T(1)};
  T a = R::el_cos(e.lo), b = R::el_cos(e.hi);
  Iv<T> r = {pad_dn(mn(a, b)), pad_up(mx(a, b))};
  if (e.lo <= T(0) && e.hi >= T(0)) r.hi = T(1);
  if (e.lo <= R::pi_hi() && e.hi >= R::pi_lo()) r.lo = T(-1);
  if (e.lo <= -R::pi_lo() && e.hi >= -R::pi_hi()) r.lo = T(-1);
  return iclamp(r, T(-1), T(1));
}
// atan2(y, x) over the rectangle y x x.  Away from the cut (negative x axis) and the origin the
// angle is monotone along every edge, so the extremes sit at corners; on the cut: [-pi, pi].
template <class T> IA_DEV Iv<T> iatan2(Iv<T> y, Iv<T> x) {
  using R = Rnd<T>;
  if (x.lo <= T(0) && y.lo <= T(0) && y.hi >= T(0)) return {-R::pi_hi(), R::pi_hi()};
  T c0 = R::el_atan2(y.lo, x.lo), c1 = R::el_atan2(y.lo, x.hi), c2 = R::el_atan2(y.hi, x.lo), c3 = R::el_atan2(y.hi, x.hi);
  Iv<T> r = {pad_dn(mn(mn(c0, c1), mn(c2, c3))), pad_up(mx(mx(c0, c1), mx(c2, c3)))};
  return iclamp(r, -R::pi_hi(), R::pi_hi());
}

}  // namespace ia
