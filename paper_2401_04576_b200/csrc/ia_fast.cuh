// ia_fast.cuh - the sign-specialised form of the residual enclosure (steps S4-S8) for the dense vote.
//
// Same expression DAG as ia_residual.cuh, same association order, same tightest directed roundings;
// what changes is how each interval product is formed.  A general product needs 8 directed
// multiplies and 6 min/max; when one factor has a known sign it needs 2 multiplies and 2 selects,
// and when both signs are known, 2 multiplies.  Signs are made known in three ways:
//   * by construction: R > 0, 1/R_Ax^2 > 0, R_Ax > 0, T^2 >= 0, u_d > 0, |delta| >= 0, squares >= 0;
//   * by three exact symmetries of the DAG (negating an interval operand negates the product
//     exactly, because rounding down -x equals minus rounding up x):
//        S_a: (lambda, z0 - z_ref, T)      -> -(...)   mirror z -> -z                     f unchanged
//        S_b: (s_Ax, c_Ax, T)              -> -(...)   the same wire described by phi_s+pi, -tau
//        S_d: (s_Ax, z0 - z_ref, dphi, T)  -> -(...)   Phi -> -Phi
//     applied per (warp, hit) so that lambda >= 0 (a = [lambda <= 0], per warp), c_Ax >= 0
//     (b = [c_Ax <= 0], per hit) and T >= 0 (d = [T < 0] + a + b).  Then z0 - z_ref flips by
//     [T<0] + b (per hit), s_Ax by [T<0] + a, sin 2Phi_Ax and dphi by [T<0] + a + b: the record below
//     stores both a-versions of those three;
//   * what is left - the sign class of s_Ax, sin 2Phi_Ax, cos 2Phi_Ax (P, N or straddling M) and of
//     c_Ax (P or M) - is the same for every thread of a block, so each of the six products that has
//     such a factor picks its form by a branch no warp diverges on; the drift sign of the two
//     passes is likewise a uniform run-time flag (three +/- sites).
// One compiled body serves every sign combination: the hot loop stays within the 32 KB
// instruction cache (a body per sign combination does not, and starves the issue ports).
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

// a >= 0, x of unknown sign
template <class T> IA_DEV Iv<T> mul_pu(Iv<T> a, Iv<T> x) {
  using R = Rnd<T>;
  return {R::mul_dn(sgn(x.lo) ? a.hi : a.lo, x.lo), R::mul_up(sgn(x.hi) ? a.lo : a.hi, x.hi)};
}
// a <= 0, x of unknown sign
template <class T> IA_DEV Iv<T> mul_nu(Iv<T> a, Iv<T> x) {
  using R = Rnd<T>;
  return {R::mul_dn(sgn(x.hi) ? a.hi : a.lo, x.hi), R::mul_up(sgn(x.lo) ? a.lo : a.hi, x.lo)};
}
template <class T> IA_DEV Iv<T> mul_pp(Iv<T> a, Iv<T> b) { return {Rnd<T>::mul_dn(a.lo, b.lo), Rnd<T>::mul_up(a.hi, b.hi)}; }
// a >= 0, b <= 0
template <class T> IA_DEV Iv<T> mul_pn(Iv<T> a, Iv<T> b) { return {Rnd<T>::mul_dn(a.hi, b.lo), Rnd<T>::mul_up(a.lo, b.hi)}; }
// m straddles 0, x of unknown sign: two candidates per endpoint
template <class T> IA_DEV Iv<T> mul_mu(Iv<T> m, Iv<T> x) {
  using R = Rnd<T>;
  return {mn(R::mul_dn(x.lo, m.hi), R::mul_dn(x.hi, m.lo)), mx(R::mul_up(x.lo, m.lo), R::mul_up(x.hi, m.hi))};
}
enum { CLS_P = 0, CLS_N = 1, CLS_M = 2 };
// a of block-uniform sign class times x of unknown sign
template <class T> IA_DEV Iv<T> mul_cu(int cls, Iv<T> a, Iv<T> x) {
  if (cls == CLS_P) return mul_pu(a, x);
  if (cls == CLS_N) return mul_nu(a, x);
  return mul_mu(a, x);
}
// scalar of compile-time sign times interval
template <int S, class T> IA_DEV Iv<T> scale_s(T c, Iv<T> a) {
  using R = Rnd<T>;
  if (S >= 0) return {R::mul_dn(c, a.lo), R::mul_up(c, a.hi)};
  return {R::mul_dn(c, a.hi), R::mul_up(c, a.lo)};
}
// square of an interval of unknown sign without branches: largest / smallest magnitude
template <class T> IA_DEV Iv<T> sqr_u(Iv<T> a) {
  using R = Rnd<T>;
  const bool c = fabs(a.lo) > fabs(a.hi);
  const T mag = c ? a.lo : a.hi, mnn = c ? a.hi : a.lo;
  const bool straddle = sgn(a.lo) != sgn(a.hi);
  const T lo2 = R::mul_dn(mnn, mnn);
  return {straddle ? T(0) : lo2, R::mul_up(mag, mag)};
}

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
};
template <> struct Dir<float> {
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
template <class T> struct Trig;
template <> struct Trig<double> {
  static IA_DEV double sin_small(double x) {
    const double s = __dmul_rn(x, x);
    double q = -2.5052108385441720e-08;               // -1/11!
    q = __fma_rn(q, s, 2.7557319223985893e-06);       //  1/9!
    q = __fma_rn(q, s, -1.9841269841269841e-04);      // -1/7!
    q = __fma_rn(q, s, 8.3333333333333332e-03);       //  1/5!
    q = __fma_rn(q, s, -1.6666666666666666e-01);      // -1/3!
    return __fma_rn(__dmul_rn(x, s), q, x);
  }
  static IA_DEV double cos_small(double x) {
    const double s = __dmul_rn(x, x);
    double q = 2.0876756987868100e-09;                //  1/12!
    q = __fma_rn(q, s, -2.7557319223985888e-07);      // -1/10!
    q = __fma_rn(q, s, 2.4801587301587302e-05);       //  1/8!
    q = __fma_rn(q, s, -1.3888888888888889e-03);      // -1/6!
    q = __fma_rn(q, s, 4.1666666666666664e-02);       //  1/4!
    q = __fma_rn(q, s, -0.5);
    return __fma_rn(q, s, 1.0);
  }
};
template <> struct Trig<float> {
  static IA_DEV float sin_small(float x) {
    const float s = __fmul_rn(x, x);
    float q = -1.9841270e-04f;
    q = __fmaf_rn(q, s, 8.3333338e-03f);
    q = __fmaf_rn(q, s, -1.6666667e-01f);
    return __fmaf_rn(__fmul_rn(x, s), q, x);
  }
  static IA_DEV float cos_small(float x) {
    const float s = __fmul_rn(x, x);
    float q = 2.4801588e-05f;
    q = __fmaf_rn(q, s, -1.3888889e-03f);
    q = __fmaf_rn(q, s, 4.1666668e-02f);
    q = __fmaf_rn(q, s, -0.5f);
    return __fmaf_rn(q, s, 1.0f);
  }
};

// ---- per-(block, hit) record in shared memory ------------------------------------------------------
enum { HIT_SKIP = 0, HIT_FORCED = 1, HIT_FAST = 2, HIT_GENERAL = 3 };

template <class T> struct HitF {
  // transformed by S_b^b S_d^(t+b) (and, in the [1] versions, additionally by the S_d that goes with S_a)
  Iv<T> Q, cA, iQ, hiQ, RA, iR, c2, T2;
  Iv<T> sA[2], s2[2], dphi[2];     // index a = 1 for warps whose lambda was negated
  T Tabs;                          // |tan tau|
  T Dlo, Dhi;
  int kind;
  int ccls, c2cls;                 // classes of cA (P or M) and c2
  int scls[2], s2cls[2];           // classes of sA[a], s2[a]
  int zflip;                       // z0 - z_ref enters negated
};

template <class T> IA_DEV int cls_of(Iv<T> a) { return a.lo >= T(0) ? CLS_P : (a.hi <= T(0) ? CLS_N : CLS_M); }

// a4 + normalisation.  Rlo_min: smallest R.lo of the grid, Lmag: largest |lambda| of the grid.
template <class T> IA_DEV void make_hitf(const XYInv<T>& v, const HitS<T>& hs, T Rlo_min, T Lmag, HitF<T>& o) {
  using Rd = Rnd<T>;
  o.Dlo = hs.Dlo; o.Dhi = hs.Dhi;
  o.Tabs = fabs(hs.Tn);
  o.Q = v.Q; o.iQ = v.iQ; o.RA = v.RA; o.iR = v.iR; o.c2 = v.c2;
  o.hiQ = {Rd::mul_rn(T(0.5), v.iQ.lo), Rd::mul_rn(T(0.5), v.iQ.hi)};      // exact scaling
  o.T2 = {Rd::mul_dn(hs.Tn, hs.Tn), Rd::mul_up(hs.Tn, hs.Tn)};             // isqr(thin(T))
  o.c2cls = cls_of(v.c2);
  const bool t = hs.Tn < T(0);
  const bool b = cls_of(v.cA) == CLS_N;
  o.cA = b ? ineg(v.cA) : v.cA;
  o.ccls = cls_of(o.cA);
  o.zflip = (t != b) ? 1 : 0;
#pragma unroll
  for (int a = 0; a < 2; ++a) {
    const bool fs = t != (a == 1);            // s_Ax flips by t + a
    const bool fd = fs != b;                  // sin 2Phi_Ax and dphi flip by t + a + b
    o.sA[a] = fs ? ineg(v.sA) : v.sA;
    o.s2[a] = fd ? ineg(v.s2) : v.s2;
    o.dphi[a] = fd ? ineg(v.dphi) : v.dphi;
    o.scls[a] = cls_of(o.sA[a]);
    o.s2cls[a] = cls_of(o.s2[a]);
  }
  if (!hs.valid) { o.kind = HIT_SKIP; return; }
  if (v.forced) { o.kind = HIT_FORCED; return; }
  // guards of the sign-known forms: R - 2D > 0, R + R_Ax - D > 0, R + delta > 0 (|delta| <= 2 D.hi as
  // long as u_d >= 1/2), u_d^2 >= 1 - 2 |T| |lambda| >= 1/2
  const bool ok = Rlo_min > T(4) * hs.Dhi && o.Tabs * Lmag <= T(0.25);
  o.kind = ok ? HIT_FAST : HIT_GENERAL;
}

// general-form sin / cos and their products with s_Ax, c_Ax for enclosures outside [-1/4, 1/4] (rare)
template <class T>
__device__ __noinline__ void trig_general(Iv<T> e, Iv<T> sA, Iv<T> cA, Iv<T>& se, Iv<T>& sce, Iv<T>& cce) {
  se = isin(e);
  const Iv<T> ce = icos(e);
  sce = imul(sA, ce);
  cce = imul(cA, ce);
}

// what a thread keeps per (hit, drift sign): S4 terms that do not depend on z0
template <class T> struct PassC {
  Iv<T> LDcA, Rm2D, G;
};

template <class T>
IA_DEV PassC<T> pass_prepare(const HitF<T>& h, bool dneg, Iv<T> L, Iv<T> R, Iv<T> L2, Iv<T> RpRA) {
  PassC<T> c;
  const Iv<T> D = dneg ? Iv<T>{-h.Dhi, -h.Dlo} : Iv<T>{h.Dlo, h.Dhi};
  const Iv<T> LD = dneg ? mul_pn(L, D) : mul_pp(L, D);
  c.LDcA = imul(LD, h.cA);
  c.Rm2D = isub(R, Iv<T>{Rnd<T>::mul_rn(T(2), D.lo), Rnd<T>::mul_rn(T(2), D.hi)});
  const Iv<T> a = iadd(h.RA, mul_pp(L2, isub(RpRA, D)));
  c.G = dneg ? mul_pn(a, D) : mul_pp(D, a);
  return c;
}

// S4-S8 for one cell and one drift sign; returns true iff 0 is in f.
// Inputs transformed: L >= 0, T = h.Tabs >= 0, cA >= 0 or M; va = the warp's a.
template <class T>
IA_DEV bool pass_vote(const HitF<T>& h, int va, bool dneg, const PassC<T>& pc, Iv<T> L, Iv<T> R, Iv<T> LR, Iv<T> T2L2,
                      Iv<T> LRdphi, Iv<T> Zr) {
  using Rd = Rnd<T>;
  const T Tn = h.Tabs;
  const Iv<T> sA = h.sA[va];
  const int scls = h.scls[va];
  // S4, z0-dependent part
  const Iv<T> zA = iadd(Zr, LRdphi);                                   // (A.8d)
  const Iv<T> zAsA = mul_cu(scls, sA, zA);
  const Iv<T> t1 = mul_pu(LR, zA);
  const Iv<T> LzA = mul_pu(L, zA);
  const Iv<T> zA2 = sqr_u(zA);
  const Iv<T> Y = mul_pu(h.iQ, iadd(zAsA, pc.LDcA));                   // Phi1 = -Y           (A.8b)
  const Iv<T> t2 = mul_cu(h.c2cls, h.c2, mul_pu(pc.Rm2D, LzA));
  const Iv<T> t3 = mul_cu(h.s2cls[va], h.s2[va], iadd(zA2, pc.G));
  const Iv<T> P2 = mul_pu(h.hiQ, iadd(isub(t1, t2), t3));              // (A.8c)
  const Iv<T> e = iadd(Iv<T>{Rd::mul_dn(Tn, -Y.hi), Rd::mul_up(Tn, -Y.lo)}, mul_pu(h.T2, P2));   // (A.8a)
  // S5
  Iv<T> se, sce, cce;
  const bool small = e.lo >= T(-0.25) && e.hi <= T(0.25);
  if (__all_sync(0xffffffffu, small)) {
    se = {pad_dn(Trig<T>::sin_small(e.lo)), pad_up(Trig<T>::sin_small(e.hi))};
    const bool c = fabs(e.lo) > fabs(e.hi);
    const T mag = c ? e.lo : e.hi, mnn = c ? e.hi : e.lo;
    const bool straddle = sgn(e.lo) != sgn(e.hi);
    const T chi = pad_up(Trig<T>::cos_small(mnn));
    const Iv<T> ce = {pad_dn(Trig<T>::cos_small(mag)), (straddle || chi > T(1)) ? T(1) : chi};   // cos > 0.96
    sce = mul_pu(ce, sA);
    cce = mul_pu(ce, h.cA);
  } else {
    trig_general(e, sA, h.cA, se, sce, cce);
  }
  const Iv<T> sinP = iclamp(mul_pu(h.iR, iadd(sce, mul_cu(h.ccls, h.cA, se))), T(-1), T(1));
  const Iv<T> cosP = iclamp(mul_pu(h.iR, isub(cce, mul_cu(scls, sA, se))), T(-1), T(1));
  // S6: u_d^2 >= 1 - 2 T max|lambda| - rounding >= 0.49 by the HIT_FAST guard: roots of normal numbers
  const T twoT = Rd::mul_rn(T(2), Tn);
  const Iv<T> u2 = iadd(iadd(iadd_s(iscale_pos(twoT, mul_pu(L, sinP)), T(1)), T2L2), mul_pp(h.T2, sqr_u(cosP)));
  T hlo, hhi;
  const T ulo = Dir<T>::sqrt_dn(u2.lo, hlo), uhi = Dir<T>::sqrt_up(u2.hi, hhi);
  // |delta| = D+ / u_d
  const Iv<T> dq = {Dir<T>::div_dn(h.Dlo, uhi, Rd::mul_rn(T(2), hhi)), Dir<T>::div_up(h.Dhi, ulo, Rd::mul_rn(T(2), hlo))};
  // S7: z = (Zr + LR (dphi + e)) - T (delta cosP), delta = -/+ dq
  const Iv<T> zz = iadd(Zr, mul_pu(LR, iadd(h.dphi[va], e)));
  const Iv<T> Tdc = iscale_pos(Tn, mul_pu(dq, cosP));
  const Iv<T> z = dneg ? iadd(zz, Tdc) : isub(zz, Tdc);
  const Iv<T> Lq = mul_pp(L, dq);                                      // |lambda delta|
  const Iv<T> zc = mul_cu(h.ccls, h.cA, z);
  const Iv<T> qs = mul_pu(Lq, sA);
  const Iv<T> ct = dneg ? iadd(zc, qs) : isub(zc, qs);                 // c^tau              (A.7b)
  // S8
  const Iv<T> Rd1 = dneg ? isub(R, dq) : iadd(R, dq);
  const Iv<T> TLq = iscale_pos(Tn, Lq);
  const Iv<T> rad = isub(isub(isub(mul_pp(Rd1, Rd1), iscale_pos(twoT, ct)), sqr_u(iscale_pos(Tn, z))), mul_pp(TLq, TLq));
  const Iv<T> f = isub(h.Q, rad);
  return !(f.lo > T(0) || f.hi < T(0));
}

}  // namespace ia
