// ia_fast.cuh - the FP64-pipe form of the residual enclosure (steps S4-S8) for the dense vote.
//
// Same expression DAG as ia_residual.cuh and the same association order.  What changes is how each
// interval product is formed.  The dense kernel is bound by the FP64 pipe and by the dependency
// latency around it (profiles/r02_pipe_probe.md: a dependent FP64 instruction issues 8 cycles after
// its producer; profiles/r01_vote_dense_fast_c1_ncu.md), and the textbook sign-case product - pick the
// partner endpoint by the sign of x, then multiply (2 DMUL + 2 ISETP + 4 FSEL) - puts a compare and a
// select between every pair of FP64 instructions.  The form below is 4 FP64 instructions and nothing else:
//
//   factor a of KNOWN sign class, kept as midpoint and radius (m, r) with [m-r, m+r] containing a,
//   times x = [x.lo, x.hi] of ANY sign:   for a >= 0
//        lower = RD( RD(m x.lo) - r |x.lo| )        upper = RU( RU(m x.hi) + r |x.hi| )
//   (g(x) = m x - r|x| is the exact lower envelope of {a' x : a' in [m-r, m+r]}; it is concave, and
//   increasing when a >= 0, so its minimum over x is at x.lo; |x| is an operand modifier of DFMA.)
//   The result encloses the true product and is at most 2 ulps wider than the tightest enclosure
//   (one rounding of (m, r), one of the inner product) - the same order as the padding of the
//   elementary functions, 4 orders below the 1e-12 knife-edge band of the parity criterion.
//   For a <= 0 the roles of x.lo and x.hi swap (the body negates m instead and flips the add/sub
//   that consumes the product); for a straddling 0 both endpoints of x are tried (prod_u).
//
// Which factors have a known class: by construction R, R_Ax^-2, R_Ax^-1, T^2, |delta|, R - 2D; by three
// exact symmetries of the DAG (negating an interval operand negates the product exactly, because
// rounding down -x equals minus rounding up x)
//        S_a: (lambda, z0 - z_ref, T)      -> -(...)   mirror z -> -z                     f unchanged
//        S_b: (s_Ax, c_Ax, T)              -> -(...)   the same wire described by phi_s+pi, -tau
//        S_d: (s_Ax, z0 - z_ref, dphi, T)  -> -(...)   Phi -> -Phi
// applied per (warp, hit) so that lambda >= 0 (a = [lambda <= 0], per warp), c_Ax >= 0 or straddling
// (b = [c_Ax <= 0], per hit) and T >= 0 (d = [T < 0] + a + b); then z0 - z_ref flips by [T<0] + b (per
// hit), s_Ax by [T<0] + a, sin 2Phi_Ax and dphi by [T<0] + a + b: the record stores both a-versions.
// What is left - the class of s_Ax (and with it of sin 2Phi_Ax), of c_Ax (P or straddling) and of
// cos 2Phi_Ax - is the same for every thread of a block and selects one of three compiled bodies per
// hit: SS = +1 (s_Ax >= 0, c_Ax >= 0), SS = -1 (s_Ax <= 0, c_Ax >= 0), SS = 0 (anything straddles:
// universal products).  cos 2Phi_Ax is dispatched inside the body (one site).  Three bodies stay
// inside the 32 KB instruction cache; a body per sign combination does not (measured, round 1).
// A hit that violates the guards in make_hitf, and a warp whose lambda cells straddle 0, take the
// general form (on the same transformed data - the symmetries are exact for it too).
//
// sqrt and division: own directed-rounding sequences (Goldschmidt from MUFU.RSQ64H, then one FMA
// residual whose sign tells on which side of the exact value the candidate lies) - results are the
// correctly rounded-down / rounded-up values, identical to IEEE directed rounding.
// sin/cos of Phi - Phi_Ax: for enclosures inside [-1/4, 1/4] Taylor polynomials with a stated bound,
// padded outward by the same relative 2^-50 as the general form; otherwise the general form.
#pragma once
#include "ia_residual.cuh"

namespace ia {

// ---- sign-known products ------------------------------------------------------------------------
// the sign bit (not "< 0"): for a zero endpoint either partner gives a zero product
IA_DEV bool sgn(double x) { return __double2hiint(x) < 0; }
IA_DEV bool sgn(float x) { return __float_as_int(x) < 0; }

// a >= 0 computed per lane (no midpoint form at hand), x of unknown sign: partner by sign of x
template <class T> IA_DEV Iv<T> mul_pu(Iv<T> a, Iv<T> x) {
  using R = Rnd<T>;
  return {R::mul_dn(sgn(x.lo) ? a.hi : a.lo, x.lo), R::mul_up(sgn(x.hi) ? a.lo : a.hi, x.hi)};
}
template <class T> IA_DEV Iv<T> mul_pp(Iv<T> a, Iv<T> b) { return {Rnd<T>::mul_dn(a.lo, b.lo), Rnd<T>::mul_up(a.hi, b.hi)}; }
// a >= 0, b <= 0
template <class T> IA_DEV Iv<T> mul_pn(Iv<T> a, Iv<T> b) { return {Rnd<T>::mul_dn(a.hi, b.lo), Rnd<T>::mul_up(a.lo, b.hi)}; }

// midpoint-radius form of a factor: [m - r, m + r] contains the interval it was made from
template <class T> struct MR { T m, r; };
template <class T> IA_DEV MR<T> to_mr(Iv<T> a) {
  using R = Rnd<T>;
  const T m = R::mul_rn(T(0.5), R::add_rn(a.lo, a.hi));
  return {m, mx(R::add_up(m, -a.lo), R::add_up(a.hi, -m))};
}
template <class T> IA_DEV MR<T> mr_neg(MR<T> a) { return {-a.m, a.r}; }
// a >= 0 (as an interval; its (m, r) hull may dip an ulp below 0, which only lowers the bound)
template <class T> IA_DEV Iv<T> prod_p(MR<T> a, Iv<T> x) {
  using R = Rnd<T>;
  return {R::fma_dn(-a.r, fabs(x.lo), R::mul_dn(a.m, x.lo)), R::fma_up(a.r, fabs(x.hi), R::mul_up(a.m, x.hi))};
}
// a of any class: lower envelope concave, upper convex -> extremes at the endpoints of x
template <class T> IA_DEV Iv<T> prod_u(MR<T> a, Iv<T> x) {
  using R = Rnd<T>;
  const T l0 = R::fma_dn(-a.r, fabs(x.lo), R::mul_dn(a.m, x.lo)), l1 = R::fma_dn(-a.r, fabs(x.hi), R::mul_dn(a.m, x.hi));
  const T h0 = R::fma_up(a.r, fabs(x.lo), R::mul_up(a.m, x.lo)), h1 = R::fma_up(a.r, fabs(x.hi), R::mul_up(a.m, x.hi));
  return {mn(l0, l1), mx(h0, h1)};
}
// SS = +1: a >= 0;  SS = -1: a <= 0, returns (-a) x;  SS = 0: a of any class, returns a x
template <int SS, class T> IA_DEV Iv<T> prod_s(MR<T> a, Iv<T> x) {
  if (SS > 0) return prod_p(a, x);
  if (SS < 0) return prod_p(mr_neg(a), x);
  return prod_u(a, x);
}
// base + sigma * t, where t = |sigma-signed term| as returned by prod_s (SS = 0: t is the term itself)
template <int SS, class T> IA_DEV Iv<T> add_s(Iv<T> base, Iv<T> t) { return SS < 0 ? isub(base, t) : iadd(base, t); }
template <int SS, class T> IA_DEV Iv<T> sub_s(Iv<T> base, Iv<T> t) { return SS < 0 ? iadd(base, t) : isub(base, t); }
// ---- fused product-and-add forms ---------------------------------------------------------------------
// base + a x and base - a x in ONE directed FMA per rounding step: RD(base.lo + m x.lo) is below the
// exact base.lo + m x.lo, and the radius term is subtracted from that, so the result is below every
// base' + a' x' - an enclosure by the same argument as prod_p, one rounding tighter than product
// followed by sum.  Operand negations and |x| are instruction modifiers.
template <class T> IA_DEV Iv<T> fma_p(MR<T> a, Iv<T> x, Iv<T> base) {            // base + a x, a >= 0
  using R = Rnd<T>;
  return {R::fma_dn(-a.r, fabs(x.lo), R::fma_dn(a.m, x.lo, base.lo)), R::fma_up(a.r, fabs(x.hi), R::fma_up(a.m, x.hi, base.hi))};
}
template <class T> IA_DEV Iv<T> fms_p(MR<T> a, Iv<T> x, Iv<T> base) {            // base - a x, a >= 0
  using R = Rnd<T>;
  return {R::fma_dn(-a.r, fabs(x.hi), R::fma_dn(-a.m, x.hi, base.lo)), R::fma_up(a.r, fabs(x.lo), R::fma_up(-a.m, x.lo, base.hi))};
}
template <class T> IA_DEV Iv<T> fma_u(MR<T> a, Iv<T> x, Iv<T> base) {            // base + a x, a of any class
  using R = Rnd<T>;
  const T l0 = R::fma_dn(-a.r, fabs(x.lo), R::fma_dn(a.m, x.lo, base.lo)), l1 = R::fma_dn(-a.r, fabs(x.hi), R::fma_dn(a.m, x.hi, base.lo));
  const T h0 = R::fma_up(a.r, fabs(x.lo), R::fma_up(a.m, x.lo, base.hi)), h1 = R::fma_up(a.r, fabs(x.hi), R::fma_up(a.m, x.hi, base.hi));
  return {mn(l0, l1), mx(h0, h1)};
}
template <class T> IA_DEV Iv<T> fms_u(MR<T> a, Iv<T> x, Iv<T> base) { return fma_u(mr_neg(a), x, base); }
// base + a x for a of class SS (+1: a >= 0, -1: a <= 0, 0: any); base - a x
template <int SS, class T> IA_DEV Iv<T> fma_s(MR<T> a, Iv<T> x, Iv<T> base) {
  if (SS > 0) return fma_p(a, x, base);
  if (SS < 0) return fms_p(mr_neg(a), x, base);
  return fma_u(a, x, base);
}
template <int SS, class T> IA_DEV Iv<T> fms_s(MR<T> a, Iv<T> x, Iv<T> base) {
  if (SS > 0) return fms_p(a, x, base);
  if (SS < 0) return fma_p(mr_neg(a), x, base);
  return fms_u(a, x, base);
}
// c >= 0 per lane times a block-uniform interval s:  SS = +1: s >= 0; -1: s <= 0, returns c (-s); 0: any
template <int SS, class T> IA_DEV Iv<T> mulpos_s(Iv<T> c, Iv<T> s) {
  if (SS > 0) return mul_pp(c, s);
  if (SS < 0) return mul_pp(c, ineg(s));
  return mul_pu(c, s);
}

// ---- comparisons kept off the FP64 pipe -----------------------------------------------------------
// The FP64 pipe is the bottleneck of the dense kernel and the ALU pipe has room (profiles/), so the
// comparisons whose operands are finite by construction are done on the bit patterns: for
// non-negative doubles the order of the values is the order of the 64-bit integers.
#ifndef IA_INT_CMP
#define IA_INT_CMP 1
#endif
#if IA_INT_CMP
IA_DEV bool abs_gt(double a, double b) {           // |a| > |b|
  // on the two 32-bit halves: written as a 64-bit mask the compiler turns the "& 0x7fff..." into DADD -RZ, |x| - two
  // instructions on the FP64 pipe per comparison, 14 per evaluation (ncu source page, round 1)
  unsigned ah, bh;
  asm("and.b32 %0, %1, 0x7fffffff;" : "=r"(ah) : "r"(__double2hiint(a)));
  asm("and.b32 %0, %1, 0x7fffffff;" : "=r"(bh) : "r"(__double2hiint(b)));
  const unsigned long long ua = ((unsigned long long)ah << 32) | (unsigned)__double2loint(a);
  const unsigned long long ub = ((unsigned long long)bh << 32) | (unsigned)__double2loint(b);
  return ua > ub;
}
IA_DEV bool nn_gt(double a, double b) { return __double_as_longlong(a) > __double_as_longlong(b); }   // a, b >= 0
IA_DEV bool is_pos(double x) { return __double_as_longlong(x) > 0; }                                 // x > 0
IA_DEV bool ge_one(double x) { return __double2hiint(x) >= 0x3ff00000; }                              // x >= 1
IA_DEV bool abs_lt_quarter(double x) { return (__double2hiint(x) & 0x7fffffff) < 0x3fd00000; }        // |x| < 1/4
#else
IA_DEV bool abs_gt(double a, double b) { return fabs(a) > fabs(b); }
IA_DEV bool nn_gt(double a, double b) { return a > b; }
IA_DEV bool is_pos(double x) { return x > 0.0; }
IA_DEV bool ge_one(double x) { return x >= 1.0; }
IA_DEV bool abs_lt_quarter(double x) { return fabs(x) < 0.25; }
#endif
IA_DEV bool abs_gt(float a, float b) { return fabsf(a) > fabsf(b); }
IA_DEV bool nn_gt(float a, float b) { return a > b; }
IA_DEV bool is_pos(float x) { return x > 0.f; }
IA_DEV bool ge_one(float x) { return x >= 1.f; }
IA_DEV bool abs_lt_quarter(float x) { return fabsf(x) < 0.25f; }

enum { CLS_P = 0, CLS_N = 1, CLS_M = 2 };
// square of an interval of unknown sign without branches: largest / smallest magnitude
template <class T> IA_DEV Iv<T> sqr_u(Iv<T> a) {
  using R = Rnd<T>;
  const bool c = abs_gt(a.lo, a.hi);
  const T mag = c ? a.lo : a.hi, mnn = c ? a.hi : a.lo;
  const bool straddle = sgn(a.lo) != sgn(a.hi);
  const T lo2 = R::mul_dn(mnn, mnn);
  return {straddle ? T(0) : lo2, R::mul_up(mag, mag)};
}
// largest / smallest magnitude endpoint and the straddle flag of an interval of unknown sign
template <class T> struct Mag { T mag, mnn; bool straddle; };
template <class T> IA_DEV Mag<T> mag_of(Iv<T> a) {
  const bool c = abs_gt(a.lo, a.hi);
  return {c ? a.lo : a.hi, c ? a.hi : a.lo, sgn(a.lo) != sgn(a.hi)};
}
// base + s a^2 and base - a^2, one FMA per endpoint (s = [s.lo, s.hi] >= 0)
template <class T> IA_DEV Iv<T> add_sqr(Iv<T> base, Iv<T> a) {
  const Mag<T> g = mag_of(a);
  return {g.straddle ? base.lo : Rnd<T>::fma_dn(g.mnn, g.mnn, base.lo), Rnd<T>::fma_up(g.mag, g.mag, base.hi)};
}
template <class T> IA_DEV Iv<T> sub_sqr(Iv<T> base, Iv<T> a) {
  const Mag<T> g = mag_of(a);
  return {Rnd<T>::fma_dn(-g.mag, g.mag, base.lo), g.straddle ? base.hi : Rnd<T>::fma_up(-g.mnn, g.mnn, base.hi)};
}
// intersection with [-1, 1] by integer tests on the high word (keeps the FP64 pipe free):
// x <= -1  <=>  hi32(x) as unsigned >= hi32(-1);  x >= 1  <=>  hi32(x) as signed >= hi32(1)
IA_DEV Iv<double> clamp_unit(Iv<double> a) {
  const bool l = (unsigned)__double2hiint(a.lo) >= 0xbff00000u, h = __double2hiint(a.hi) >= 0x3ff00000;
  Iv<double> r = {l ? -1.0 : a.lo, h ? 1.0 : a.hi};
  // opaque to the compiler: it otherwise hoists the |x| of a later DFMA operand above the select as DADD -RZ, |x| -
  // an FP64-pipe instruction where an operand modifier does the same for nothing
  asm("" : "+d"(r.lo), "+d"(r.hi));
  return r;
}
IA_DEV Iv<float> clamp_unit(Iv<float> a) {
  const bool l = (unsigned)__float_as_int(a.lo) >= 0xbf800000u, h = __float_as_int(a.hi) >= 0x3f800000;
  return {l ? -1.0f : a.lo, h ? 1.0f : a.hi};
}
// cos Phi >= 0 for both drift signs: then cos^2 needs no magnitude sort and the partners of its endpoints in
// T delta cos Phi are fixed.  After the normalisation c_Ax >= 0 this holds for 95-97 % of the warp-evaluations on C1 / C4
// (measured); the kernels test it per warp and skip ~40 compare/select instructions.  (The upper clamps at +-1 are
// active in 40 % of them - sin Phi_Ax, cos Phi_Ax and 1/R_Ax are enclosed separately over the xy cell - and stay.)
IA_DEV int hiw(double x) { return __double2hiint(x); }
IA_DEV int hiw(float x) { return __float_as_int(x); }
template <class T> IA_DEV bool cos_nonneg(const Iv<T> (&cosP)[2]) { return (hiw(cosP[0].lo) | hiw(cosP[1].lo)) >= 0; }
// x.hi := min(x.hi, 1), lower endpoint untouched
IA_DEV Iv<double> clamp_hi(Iv<double> a) {
  const bool h = __double2hiint(a.hi) >= 0x3ff00000;
  Iv<double> r = {a.lo, h ? 1.0 : a.hi};
  asm("" : "+d"(r.hi));
  return r;
}
IA_DEV Iv<float> clamp_hi(Iv<float> a) { return {a.lo, __float_as_int(a.hi) >= 0x3f800000 ? 1.0f : a.hi}; }
IA_DEV Iv<double> clamp_lo(Iv<double> a) {
  const bool l = (unsigned)__double2hiint(a.lo) >= 0xbff00000u;
  Iv<double> r = {l ? -1.0 : a.lo, a.hi};
  asm("" : "+d"(r.lo));
  return r;
}
IA_DEV Iv<float> clamp_lo(Iv<float> a) { return {(unsigned)__float_as_int(a.lo) >= 0xbf800000u ? -1.0f : a.lo, a.hi}; }

// ---- directed square root and division ----------------------------------------------------------
template <class T> struct Dir;
template <> struct Dir<double> {
  static IA_DEV double next_up(double x) { return __longlong_as_double(__double_as_longlong(x) + 1); }    // x > 0
  static IA_DEV double next_dn(double x) { return __longlong_as_double(__double_as_longlong(x) - 1); }    // x > 0
  // sqrt of x in [2^-500, 2^500]: g = candidate within 1/2 ulp (+2^-80), h ~ 1/(2 sqrt x) to 2^-40
  static IA_DEV void sqrt_core(double x, double& g, double& h) {
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    g = __dmul_rn(x, y);
    h = __dmul_rn(0.5, y);
    double r = __fma_rn(-h, g, 0.5);
    g = __fma_rn(g, r, g);
    h = __fma_rn(h, r, h);
    r = __fma_rn(-h, g, 0.5);
    g = __fma_rn(g, r, g);
    h = __fma_rn(h, r, h);
    const double d = __fma_rn(-g, g, x);
    g = __fma_rn(d, h, g);
  }
  // both directed roots of one argument's enclosure endpoints are needed separately; each returns
  // also h for the division that follows
  static IA_DEV double sqrt_dn(double x, double& h) {
    double g;
    sqrt_core(x, g, h);
    const double d = __fma_rn(-g, g, x);       // sign of x - g^2 is exact
    return d < 0.0 ? next_dn(g) : g;
  }
  static IA_DEV double sqrt_up(double x, double& h) {
    double g;
    sqrt_core(x, g, h);
    const double d = __fma_rn(-g, g, x);
    return d > 0.0 ? next_up(g) : g;
  }
  // a / b for a >= 0, b > 0, given y0 ~ 1/b to better than 2^-30
  static IA_DEV double div_core(double a, double b, double y0) {
    double e = __fma_rn(-b, y0, 1.0);
    double y = __fma_rn(y0, e, y0);
    e = __fma_rn(-b, y, 1.0);
    y = __fma_rn(y, e, y);
    double q = __dmul_rn(a, y);
    const double r = __fma_rn(-b, q, a);
    return __fma_rn(r, y, q);
  }
  static IA_DEV double div_dn(double a, double b, double y0) {
    const double q = div_core(a, b, y0);
    const double d = __fma_rn(-b, q, a);       // sign of a - b q is exact
    return (d < 0.0) ? next_dn(q) : q;
  }
  static IA_DEV double div_up(double a, double b, double y0) {
    const double q = div_core(a, b, y0);
    const double d = __fma_rn(-b, q, a);
    return (d > 0.0) ? (q > 0.0 ? next_up(q) : 4.9406564584124654e-324) : q;
  }
  // 1/sqrt(x) for x in [2^-2, 2^2], relative error below 2^-51.  y0 = MUFU.RSQ64H (relative error e0
  // < 2^-20: 1 - x y0^2 = r, |r| < 2^-19); 1/sqrt(x) = y0 (1-r)^(-1/2) = y0 (1 + r/2 + 3r^2/8 + 5r^3/16 ...):
  // truncation after r^2 leaves 5/16 |r|^3 < 2^-58; rounding: t = x y0 (2^-53 relative, carried into r
  // as 2^-53 absolute, halved), the final FMA (2^-53): together < 2^-52 + 2^-58.
  static IA_DEV double rsqrt_near(double x) {
    double y0;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y0) : "d"(x));
    const double t = __dmul_rn(x, y0);
    const double r = __fma_rn(-t, y0, 1.0);
    const double p = __fma_rn(0.375, r, 0.5);
    return __fma_rn(__dmul_rn(y0, r), p, y0);
  }
  // enclosure of D+ / sqrt(u2): 1/sqrt is decreasing; the relative 2^-50 padding of D+ (DloP, DhiP)
  // covers the 2^-51 of rsqrt_near, the product is rounded outward
  template <class H> static IA_DEV Iv<double> d_over_sqrt(const H& h, Iv<double> u2) {
    return {__dmul_rd(h.DloP, rsqrt_near(u2.hi)), __dmul_ru(h.DhiP, rsqrt_near(u2.lo))};
  }
};
template <> struct Dir<float> {
  // 1/sqrt(x) for x in [2^-2, 2^2], relative error below 2^-23: MUFU.RSQ (2^-22) and one third-order step
  static IA_DEV float rsqrt_near(float x) {
    float y0;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y0) : "f"(x));
    const float t = __fmul_rn(x, y0);
    const float r = __fmaf_rn(-t, y0, 1.0f);
    const float p = __fmaf_rn(0.375f, r, 0.5f);
    return __fmaf_rn(__fmul_rn(y0, r), p, y0);
  }
  // as in double: D+ padded outward by the relative 2^-21 covers the error of rsqrt_near; no library division
  // or square root (two calls with slow paths per endpoint)
  template <class H> static IA_DEV Iv<float> d_over_sqrt(const H& h, Iv<float> u2) {
    return {__fmul_rd(h.DloP, rsqrt_near(u2.hi)), __fmul_ru(h.DhiP, rsqrt_near(u2.lo))};
  }
  static IA_DEV float sqrt_dn(float x, float& h) { h = 0.f; return __fsqrt_rd(x); }
  static IA_DEV float sqrt_up(float x, float& h) { h = 0.f; return __fsqrt_ru(x); }
  static IA_DEV float div_dn(float a, float b, float) { return __fdiv_rd(a, b); }
  static IA_DEV float div_up(float a, float b, float) { return __fdiv_ru(a, b); }
};

// ---- sin / cos on [-1/4, 1/4] ---------------------------------------------------------------------
// Taylor polynomials in Horner form (round-to-nearest FMAs).  Truncation: |x| <= 2^-2 gives
// |x|^13/13! < 2.5e-18 |x| for sin (terms to x^11) and x^14/14! < 4.2e-20 for cos (terms to x^12);
// rounding: the last operations are x + x^3 q and 1 - x^2 r with |x^3 q| <= |x|/96, |x^2 r| <= 1/32,
// so the total error stays below 1 ulp of the result - well inside the relative pad 2^-50 (4..8 ulps).
// Float: terms to x^7 / x^8, truncation < 1e-11, pad 2^-21.
// The double coefficients sit in constant memory: a DFMA takes c[bank][offset] as an operand directly, whereas literals
// are rebuilt in uniform registers (two UMOV each) on every evaluation - there are not enough of them to keep 11 doubles.
//                                        -1/11!                   1/9!                    -1/7!                    1/5!                    -1/3!
static __constant__ double IA_SIN_C[5] = {-2.5052108385441720e-08, 2.7557319223985893e-06, -1.9841269841269841e-04, 8.3333333333333332e-03,
                                          -1.6666666666666666e-01};
//                                        1/12!                   -1/10!                   1/8!                    -1/6!                    1/4!
static __constant__ double IA_COS_C[6] = {2.0876756987868100e-09, -2.7557319223985888e-07, 2.4801587301587302e-05, -1.3888888888888889e-03,
                                          4.1666666666666664e-02, -0.5};
// Medium range, |x| < 1 (round 2; the float form is in Trig<float>): terms to x^19 / x^20 - truncation x^21/21! < 2e-20 |x| and x^22/22! < 1e-21;
// rounding, with u = 2^-53: sin = x + x^3 q: |error| <= 0.84 u |x| (x^3 q, |q| <= 1/6) + u |sin x| <= 2 u |sin x| as
// sin x >= 0.84 |x|; cos = 1 + x^2 r: |error| <= 2.1 u (x^2 r with |r| <= 1/2, last two Horner steps, the final FMA)
// <= 3.9 u cos x as cos x >= 0.54 - both inside the relative pad 2^-50 = 8 u.  On the 8^5 start grid of a refinement 11 %
// of the warp-evaluations have a lane with |e| in [1/4, 1) and took the general form for it (library sin/cos and two
// general products: 720 warp-instructions against 100 here; profiles/).
//                                        -1/19!                  1/17!                   -1/15!                  1/13!
static __constant__ double IA_SIN_M[9] = {-8.22063524662433e-18, 2.8114572543455206e-15, -7.647163731819816e-13, 1.6059043836821613e-10,
//                                        -1/11!                  1/9!                    -1/7!                   1/5!                  -1/3!
                                          -2.505210838544172e-08, 2.7557319223985893e-06, -0.0001984126984126984, 0.008333333333333333,
                                          -0.16666666666666666};
//                                         1/20!                  -1/18!                   1/16!                  -1/14!
static __constant__ double IA_COS_M[10] = {4.110317623312165e-19, -1.5619206968586225e-16, 4.779477332387385e-14, -1.1470745597729725e-11,
//                                         1/12!                 -1/10!                  1/8!                  -1/6!                   1/4!
                                           2.08767569878681e-09, -2.755731922398589e-07, 2.48015873015873e-05, -0.001388888888888889,
                                           0.041666666666666664, -0.5};
template <class T> struct Trig;
template <> struct Trig<double> {
  static IA_DEV double sin_medium(double x, double s) {
    double q = __fma_rn(IA_SIN_M[0], s, IA_SIN_M[1]);
#pragma unroll
    for (int k = 2; k < 9; ++k) q = __fma_rn(q, s, IA_SIN_M[k]);
    return __fma_rn(__dmul_rn(x, s), q, x);
  }
  static IA_DEV double cos_medium(double s) {
    double q = __fma_rn(IA_COS_M[0], s, IA_COS_M[1]);
#pragma unroll
    for (int k = 2; k < 10; ++k) q = __fma_rn(q, s, IA_COS_M[k]);
    return __fma_rn(q, s, 1.0);
  }
  static IA_DEV double sqr(double x) { return __dmul_rn(x, x); }
  static IA_DEV double sin_small(double x, double s) {
    double q = __fma_rn(IA_SIN_C[0], s, IA_SIN_C[1]);
    q = __fma_rn(q, s, IA_SIN_C[2]);
    q = __fma_rn(q, s, IA_SIN_C[3]);
    q = __fma_rn(q, s, IA_SIN_C[4]);
    return __fma_rn(__dmul_rn(x, s), q, x);
  }
  static IA_DEV double cos_small(double s) {
    double q = __fma_rn(IA_COS_C[0], s, IA_COS_C[1]);
    q = __fma_rn(q, s, IA_COS_C[2]);
    q = __fma_rn(q, s, IA_COS_C[3]);
    q = __fma_rn(q, s, IA_COS_C[4]);
    q = __fma_rn(q, s, IA_COS_C[5]);
    return __fma_rn(q, s, 1.0);
  }
};
template <> struct Trig<float> {
  // medium range in float: terms to x^11 / x^12 (truncation x^13/13! < 1.7e-10, x^14/14! < 1.2e-11 against 2^-24 = 6e-8); the
  // rounding bound is the double one with u = 2^-24: 2 u |sin x|, 3.9 u cos x, inside the relative pad 2^-21 = 8 u
  static IA_DEV float sm(int k) { const float c[5] = {-2.5052108e-08f, 2.7557319e-06f, -1.9841270e-04f, 8.3333338e-03f, -1.6666667e-01f}; return c[k]; }
  static IA_DEV float cm(int k) { const float d[6] = {2.0876757e-09f, -2.7557319e-07f, 2.4801588e-05f, -1.3888889e-03f, 4.1666668e-02f, -0.5f}; return d[k]; }
  static IA_DEV float sin_medium(float x, float s) {
    float q = __fmaf_rn(sm(0), s, sm(1));
#pragma unroll
    for (int k = 2; k < 5; ++k) q = __fmaf_rn(q, s, sm(k));
    return __fmaf_rn(__fmul_rn(x, s), q, x);
  }
  static IA_DEV float cos_medium(float s) {
    float q = __fmaf_rn(cm(0), s, cm(1));
#pragma unroll
    for (int k = 2; k < 6; ++k) q = __fmaf_rn(q, s, cm(k));
    return __fmaf_rn(q, s, 1.0f);
  }
  static IA_DEV float sqr(float x) { return __fmul_rn(x, x); }
  static IA_DEV float sin_small(float x, float s) {
    float q = -1.9841270e-04f;
    q = __fmaf_rn(q, s, 8.3333338e-03f);
    q = __fmaf_rn(q, s, -1.6666667e-01f);
    return __fmaf_rn(__fmul_rn(x, s), q, x);
  }
  static IA_DEV float cos_small(float s) {
    float q = 2.4801588e-05f;
    q = __fmaf_rn(q, s, -1.3888889e-03f);
    q = __fmaf_rn(q, s, 4.1666668e-02f);
    q = __fmaf_rn(q, s, -0.5f);
    return __fmaf_rn(q, s, 1.0f);
  }
};

// sin and cos over e inside [-1/4, 1/4]: sin is increasing there, cos decreases in |e|.  The squares
// serve both polynomials; |e.lo| > |e.hi| is read off them (equal squares give equal cosines).
template <class T> IA_DEV void trig_small(Iv<T> e, Iv<T>& se, Iv<T>& ce) {
  const T s0 = Trig<T>::sqr(e.lo), s1 = Trig<T>::sqr(e.hi);
  se = {pad_dn(Trig<T>::sin_small(e.lo, s0)), pad_up(Trig<T>::sin_small(e.hi, s1))};
  const T c0 = Trig<T>::cos_small(s0), c1 = Trig<T>::cos_small(s1);
  const bool c = nn_gt(s0, s1);
  const bool straddle = sgn(e.lo) != sgn(e.hi);
  const T chi = pad_up(c ? c1 : c0);
  ce = {pad_dn(c ? c0 : c1), (straddle || ge_one(chi)) ? T(1) : chi};   // cos > 0.96
}

// the same over e inside (-1, 1) (prim op 18 / 19; the kernels use the quad form in ia_fastq.cuh)
template <class T> IA_DEV void trig_medium(Iv<T> e, Iv<T>& se, Iv<T>& ce) {
  const T s0 = Trig<T>::sqr(e.lo), s1 = Trig<T>::sqr(e.hi);
  se = {pad_dn(Trig<T>::sin_medium(e.lo, s0)), pad_up(Trig<T>::sin_medium(e.hi, s1))};
  const T c0 = Trig<T>::cos_medium(s0), c1 = Trig<T>::cos_medium(s1);
  const bool c = nn_gt(s0, s1);
  const bool straddle = sgn(e.lo) != sgn(e.hi);
  const T chi = pad_up(c ? c1 : c0);
  ce = {pad_dn(c ? c0 : c1), (straddle || ge_one(chi)) ? T(1) : chi};
}

// ---- the FP32 fast form as a floating-point filter ---------------------------------------------------
// The sign-specialised form and the general form enclose the same function but round differently (fused FMAs, midpoint-
// radius products, re-associated constants): their endpoints of f differ by a few ulps of the residual's scale
// (max(R_Ax^2, (R + d_Ax)^2); at a sign change of f both are equal).  In double that is 1e-15 relative, 3 orders inside
// the 1e-12 knife-edge band of the parity criterion, and changes no decision in practice.  In float it is 1e-6 of f's
// scale against cells whose f varies by 1e-3 of it at the deep refinement levels: one vote in 10^4 flipped, and C3's
// kept boxes differed from the oracle's in 1 event of 1,024.  So the float fast form only DECIDES when both endpoints of
// one sign's f are further than `band` = 2^-20 * R_Ax^2.hi (8 ulps of the scale; the two forms differ by at most
// 5 roundings of scale-sized terms, tests/test_gpu_parity.py checks <= 4 ulps on 10^6 evaluations) from zero, or
// when both signs exclude by that margin; anything closer is re-evaluated in the general form, which does the
// oracle's arithmetic operation for operation.
template <class T> struct Filter;
template <> struct Filter<double> { static constexpr bool on = false; static IA_DEV double rel() { return 0.0; } };
template <> struct Filter<float> { static constexpr bool on = true; static IA_DEV float rel() { return 0x1p-20f; } };
// bit 0: the vote; bit 1: ambiguous (float only) - the caller re-takes the decision in the general form
template <class T> IA_DEV unsigned decide(const Iv<T> (&f)[2], T band) {
  // f.hi is a round-up sum of finite terms: never -0, never NaN here, so "f.hi < 0" is its sign bit (no DSETP)
  const bool v0 = !(is_pos(f[0].lo) || sgn(f[0].hi)), v1 = !(is_pos(f[1].lo) || sgn(f[1].hi));
  unsigned r = (v0 || v1) ? 1u : 0u;
  if (Filter<T>::on) {
    const bool in0 = f[0].lo < -band && f[0].hi > band, in1 = f[1].lo < -band && f[1].hi > band;
    const bool out0 = f[0].lo > band || f[0].hi < -band, out1 = f[1].lo > band || f[1].hi < -band;
    if (!(in0 || in1 || (out0 && out1))) r |= 2u;
  }
  return r;
}

// ---- per-(block, hit) record in shared memory ------------------------------------------------------
// HIT_FAST_P / _N / _U: the three bodies (SS = +1, -1, 0)
enum { HIT_SKIP = 0, HIT_FORCED = 1, HIT_FAST_P = 2, HIT_FAST_N = 3, HIT_FAST_U = 4, HIT_GENERAL = 5 };

template <class T> struct __align__(16) HitF {
  // transformed by S_b^b S_d^(t+b) (and, in the [1] versions, additionally by the S_d that goes with S_a);
  // (m, r) forms carry the true sign of the factor in m
  Iv<T> Q, cA, T2, RA;
  MR<T> cAm, iRm, c2m;
  MR<T> TiQm, T2hiQm, cA2Tm;       // T/Q, T^2/(2Q), 2T c_Ax: the thin scalar folded into the block constant
  Iv<T> sA[2], dphi[2];            // index a = 1 for warps whose lambda was negated
  Iv<T> sA2T[2];                   // 2T s_Ax
  Iv<T> sA2[2];                    // 2 s_Ax (exact)
  MR<T> sAm[2], s2m[2];
  Iv<T> iQ, iR, c2, s2[2];         // interval forms, general fallback only
  // scalars after the pairs: every Iv / MR above sits on a 16-byte (8-byte in float) boundary, which the vector
  // ld.shared of HitLds (ia_fastq.cuh) needs
  T cAabs, sAabs, c2abs, s2abs, dphiabs, iQhi, RAhi, dm;   // magnitudes for the crude enclosure (prefilter, IA_FLAG_PREFILTER)
  T twoT;                          // 2 |tan tau| (exact)
  T Tabs;                          // |tan tau|
  T Dlo, Dhi;
  T DloP, DhiP;                    // D+ padded outward by 2^-50 (2^-21): absorbs the error of rsqrt_near
  T band;                          // FP32 filter: decisions with an endpoint of f within +-band of 0 are re-taken in the general form
  int kind[2];                     // per a
  int c2cls;
  int zflip;                       // z0 - z_ref enters negated
};

template <class T> IA_DEV int cls_of(Iv<T> a) { return a.lo >= T(0) ? CLS_P : (a.hi <= T(0) ? CLS_N : CLS_M); }

// a4 + normalisation.  Rlo_min: smallest R.lo of the grid, Lmag: largest |lambda| of the grid.
template <class T> IA_DEV void make_hitf(const XYInv<T>& v, const HitS<T>& hs, T Rlo_min, T Lmag, HitF<T>& o) {
  using Rd = Rnd<T>;
  o.Dlo = hs.Dlo; o.Dhi = hs.Dhi;
  o.Tabs = fabs(hs.Tn);
  o.Q = v.Q; o.iQ = v.iQ; o.RA = v.RA; o.iR = v.iR; o.c2 = v.c2;
  o.iRm = to_mr(v.iR);
  o.c2m = to_mr(v.c2);
  o.T2 = {Rd::mul_dn(hs.Tn, hs.Tn), Rd::mul_up(hs.Tn, hs.Tn)};              // isqr(thin(T))
  o.TiQm = to_mr(iscale_pos(o.Tabs, v.iQ));
  o.T2hiQm = to_mr(mul_pp(o.T2, Iv<T>{Rd::mul_rn(T(0.5), v.iQ.lo), Rd::mul_rn(T(0.5), v.iQ.hi)}));
  o.DloP = Rd::fma_dn(-hs.Dlo, Rd::pad_rel(), hs.Dlo);
  o.DhiP = Rd::fma_up(hs.Dhi, Rd::pad_rel(), hs.Dhi);
  o.c2cls = cls_of(v.c2);
  o.band = Rd::mul_up(v.Q.hi, Filter<T>::rel());
  o.cAabs = mx(fabs(v.cA.lo), fabs(v.cA.hi)); o.sAabs = mx(fabs(v.sA.lo), fabs(v.sA.hi));
  o.c2abs = mx(fabs(v.c2.lo), fabs(v.c2.hi)); o.s2abs = mx(fabs(v.s2.lo), fabs(v.s2.hi));
  o.dphiabs = mx(fabs(v.dphi.lo), fabs(v.dphi.hi));
  o.iQhi = v.iQ.hi; o.RAhi = v.RA.hi;
  o.dm = Rd::mul_up(o.DhiP, T(1.4143));                 // |delta| = D/u_d <= D.hi / sqrt(1/2): u_d^2 >= 1 - 2 |T| max|lambda| >= 1/2 by the guard
  const bool t = hs.Tn < T(0);
  const bool b = cls_of(v.cA) == CLS_N;
  o.cA = b ? ineg(v.cA) : v.cA;
  o.cAm = to_mr(o.cA);
  const T twoT = Rd::mul_rn(T(2), o.Tabs);
  o.cA2Tm = to_mr(iscale_pos(twoT, o.cA));
  o.twoT = twoT;
  const int ccls = cls_of(o.cA);
  o.zflip = (t != b) ? 1 : 0;
  // guards of the sign-known forms: R - 2D > 0, R + R_Ax - D > 0, R + delta > 0 (|delta| <= 2 D.hi as
  // long as u_d >= 1/2), u_d^2 >= 1 - 2 |T| |lambda| >= 1/2
  const bool ok = Rlo_min > T(4) * hs.Dhi && o.Tabs * Lmag <= T(0.25);
#pragma unroll
  for (int a = 0; a < 2; ++a) {
    const bool fs = t != (a == 1);            // s_Ax flips by t + a
    const bool fd = fs != b;                  // sin 2Phi_Ax and dphi flip by t + a + b
    o.sA[a] = fs ? ineg(v.sA) : v.sA;
    o.s2[a] = fd ? ineg(v.s2) : v.s2;
    o.dphi[a] = fd ? ineg(v.dphi) : v.dphi;
    o.sAm[a] = to_mr(o.sA[a]);
    o.sA2T[a] = iscale_pos(twoT, o.sA[a]);
    o.sA2[a] = {Rd::mul_rn(T(2), o.sA[a].lo), Rd::mul_rn(T(2), o.sA[a].hi)};
    o.s2m[a] = to_mr(o.s2[a]);
    const int scls = cls_of(o.sA[a]), s2cls = cls_of(o.s2[a]);
    int kind = HIT_FAST_U;
    if (ccls == CLS_P && scls == CLS_P && s2cls == CLS_P) kind = HIT_FAST_P;
    if (ccls == CLS_P && scls == CLS_N && s2cls == CLS_N) kind = HIT_FAST_N;
    if (!ok) kind = HIT_GENERAL;
    if (v.forced) kind = HIT_FORCED;
    if (!hs.valid) kind = HIT_SKIP;
    o.kind[a] = kind;
  }
}

// general-form sin / cos and their products with s_Ax, c_Ax for enclosures outside [-1/4, 1/4] (rare)
// (returned by value: with reference parameters the callers' se/sce/cce lived in local memory and the common path
// stored all six intervals there on every evaluation - 8 STL.128 per evaluation in the round-1 profile)
template <class T> struct Trig3 { Iv<T> se, sce, cce; };
template <class T>
__device__ __noinline__ Trig3<T> trig_general(Iv<T> e, Iv<T> sA, Iv<T> cA) {
  Trig3<T> r;
  r.se = isin(e);
  const Iv<T> ce = icos(e);
  r.sce = imul(sA, ce);
  r.cce = imul(cA, ce);
  return r;
}

// what a thread keeps per (R, lambda) pair
template <class T> struct PairC {
  Iv<T> L, R;          // lambda >= 0 after S_a, R > 0
  MR<T> Lm, LRm;       // midpoint forms of lambda and lambda R
  Iv<T> L2;            // lambda^2
};
// ---- crude enclosure of f over a whole z0 tile (prefilter, IA_FLAG_PREFILTER) --------------------------------------------
// Condition (4) asks whether 0 is in the interval extension F of f = R_Ax^2 - (R + d_Ax)^2.  Any enclosure G of F answers
// "no" safely: 0 not in G implies 0 not in F ("if the condition is false the solution is not in the
// voxel" holds for every valid enclosure; the paper's own disk pre-filter L64-72 is such a cheaper test).  G here bounds,
// by magnitudes, every step of S4-S8 for both drift signs and all z0 cells of the block's tile at once:
//   |zA| <= zeta + LR |dphi|                 zeta = largest |z0 - z_ref| of the tile
//   |e|  <= T |P1| + T^2 |P2|                 products and sums of intervals bounded by products and sums of magnitudes
//   |z|  <= zeta + LR (|dphi| + |e|) + T dm   |cos Phi| <= 1 after the clamp, |delta| <= dm = 1.4143 D.hi (u_d^2 >= 1/2)
//   |c^tau| <= |z| |c_Ax| + lambda dm |s_Ax|
//   rad = (R + delta)^2 - S,  S = 2T c^tau + (T z)^2 + (T lambda delta)^2 in [-S1, S2]
//   rad in [(R.lo - dm)^2 - S2, (R.hi + dm)^2 + S1]   ->   excluded iff Q.lo > rad.hi or Q.hi < rad.lo
// Upper bounds are rounded up, the lower one down, and both are pushed out by a relative `slack` of the scale, far more
// than the roundings of the fine evaluation widen ITS enclosure.  On C4 (64^5) the fine enclosure keeps 0 for 5 % of the
// (cell, hit) pairs; this bound excludes most of the rest for the cost of ~40 FP64 instructions per (pair, hit, 16 cells).
// A warp skips a hit only if every lane is excluded; otherwise all lanes take the fine evaluation as before, so the votes
// are those of the fine evaluation in every case (tests compare both modes cell by cell).
template <class T> struct Crude;
template <> struct Crude<double> { static IA_DEV double slack() { return 0x1p-40; } };
template <> struct Crude<float> { static IA_DEV float slack() { return 0x1p-12f; } };
template <class T> IA_DEV bool crude_excludes(const HitF<T>& h, const PairC<T>& p, T zeta) {
  using R = Rnd<T>;
  const T Lh = p.L.hi, Rl = p.R.lo, Rh = p.R.hi, Dh = h.Dhi, Tn = h.Tabs, dm = h.dm;
  const T LRh = R::add_up(p.LRm.m, p.LRm.r);
  const T zAm = R::fma_up(LRh, h.dphiabs, zeta);
  const T P1 = R::mul_up(R::fma_up(zAm, h.sAabs, R::mul_up(R::mul_up(Lh, Dh), h.cAabs)), h.iQhi);
  const T a1 = R::mul_up(LRh, zAm);
  const T a2 = R::mul_up(R::mul_up(R::mul_up(Lh, zAm), R::fma_up(T(2), Dh, Rh)), h.c2abs);
  const T g = R::fma_up(R::mul_up(Lh, Lh), R::add_up(R::add_up(Rh, h.RAhi), Dh), h.RAhi);
  const T a3 = R::mul_up(R::fma_up(zAm, zAm, R::mul_up(Dh, g)), h.s2abs);
  const T P2 = R::mul_up(T(0.5), R::mul_up(R::add_up(R::add_up(a1, a2), a3), h.iQhi));
  const T E = R::fma_up(h.T2.hi, P2, R::mul_up(Tn, P1));
  const T zm = R::fma_up(Tn, dm, R::fma_up(LRh, R::add_up(h.dphiabs, E), zeta));
  const T Ldm = R::mul_up(Lh, dm);
  const T S1 = R::mul_up(h.twoT, R::fma_up(zm, h.cAabs, R::mul_up(Ldm, h.sAabs)));
  const T Tz = R::mul_up(Tn, zm), TLd = R::mul_up(Tn, Ldm);
  const T S2 = R::fma_up(TLd, TLd, R::fma_up(Tz, Tz, S1));
  const T rp = R::add_up(Rh, dm), rm = R::add_dn(Rl, -dm);
  T rad_hi = R::fma_up(rp, rp, S1);
  T rad_lo = R::fma_dn(rm, rm, -S2);
  const T m = R::mul_up(mx(rad_hi, h.Q.hi), Crude<T>::slack());
  rad_hi = R::add_up(rad_hi, m);
  rad_lo = R::add_dn(rad_lo, -m);
  return rm > T(0) && (h.Q.lo > rad_hi || h.Q.hi < rad_lo);
}

// ... per (pair, hit)
template <class T> struct HitP {
  Iv<T> LRdphi, T2L2, RpRA;      // lambda R dphi;  1 + T^2 lambda^2;  R + R_Ax
  MR<T> TL2m;                    // (2T) lambda in midpoint form
};

template <class T> IA_DEV HitP<T> hit_prepare(const HitF<T>& h, int va, const PairC<T>& p) {
  return {prod_p(p.LRm, h.dphi[va]), iadd_s(mul_pp(h.T2, p.L2), T(1)), iadd(p.R, h.RA), to_mr(iscale_pos(h.twoT, p.L))};
}

// The evaluation itself (S4-S8 for both drift signs of one cell) is pass_vote_q / pass_vote_qr of ia_fastq.cuh.
// Round 1 went through four earlier forms of it - products followed by sums, several z0 cells side by side, fused
// directed FMAs one sign at a time, both signs without instruction ordering - which the git history keeps
// (commits 94cbacd ... d7c361e); the measured steps are in DESIGN.md section 12.

// ---- both drift signs side by side ------------------------------------------------------------------
// The two signs of one (cell, hit) are independent dependency chains that share zA, t1 and the
// magnitude sort of zA.  Written side by side they give the FP64 pipe four independent instructions
// per step (two endpoints x two signs), which covers its 8-cycle dependent-issue latency from inside
// one warp (profiles/r02_pipe_probe.md).
// D- = -D+ exactly, hence lambda D- c_Ax = -(lambda D+ c_Ax) exactly (negation commutes with directed
// rounding); G and K differ between the signs and are kept for both.
template <class T> struct Pass2 {
  Iv<T> LDcA;          // lambda D+ c_Ax
  Iv<T> G[2];          // D (R_Ax + lambda^2 (R + R_Ax - D)) for D+, D-
  MR<T> Km[2];         // (lambda (R - 2D)) cos 2Phi_Ax for D+, D-
};
template <class T> IA_DEV Pass2<T> pass_prepare2(const HitF<T>& h, const PairC<T>& p, const HitP<T>& hp) {
  using Rd = Rnd<T>;
  Pass2<T> c;
  const Iv<T> D = {h.Dlo, h.Dhi}, Dn = {-h.Dhi, -h.Dlo};
  c.LDcA = imul(mul_pp(p.L, D), h.cA);
  const Iv<T> D2 = {Rd::mul_rn(T(2), D.lo), Rd::mul_rn(T(2), D.hi)};
  c.Km[0] = to_mr(mul_pu(mul_pp(p.L, isub(p.R, D2)), h.c2));
  c.Km[1] = to_mr(mul_pu(mul_pp(p.L, iadd(p.R, D2)), h.c2));
  c.G[0] = mul_pp(D, iadd(h.RA, mul_pp(p.L2, isub(hp.RpRA, D))));
  c.G[1] = mul_pn(iadd(h.RA, mul_pp(p.L2, isub(hp.RpRA, Dn))), Dn);
  return c;
}

}  // namespace ia
