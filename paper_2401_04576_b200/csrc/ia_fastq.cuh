// ia_fastq.cuh - S4-S8 for both drift signs of one (cell, hit), scheduled for the FP64 pipe of sm_100a.
//
// Why this file exists (measured on B200, profiles/r02_pipe_probe.md and DESIGN.md section 6.1): a
// sub-partition issues one FP64 warp instruction per 2 cycles, a dependent one 8 cycles after its
// producer, and the dense kernel runs 4 warps per sub-partition (128 registers per thread), each of
// which stalls on FP64 -> compare/select -> FP64 dependencies.  Four independent FP64 instructions in a
// row from ONE warp keep the pipe busy through such a stall of the other warps.  The two endpoints of
// an interval and the two drift signs of an evaluation are four independent chains, so every step of
// the DAG is written here as a "quad": the four first-stage instructions, then the four second-stage
// ones.  The directed operations are volatile inline PTX so that the compiler keeps that order (it
// otherwise serialises each endpoint chain to save registers: 4 dependent DFMA in a row, the other
// endpoint 60 instructions later).  Measured: C1 37.5 -> 32.4 ms.
//
// The arithmetic is that of ia_fast.cuh (fused forms, same DAG, same association order): only the
// instruction order differs.
#pragma once
#include <cstddef>

#include "ia_fast.cuh"

namespace ia {

// ---- order-preserving directed operations ---------------------------------------------------------
template <class T> struct VR;
template <> struct VR<double> {
#define IA_VOP2(name, ptx) \
  static IA_DEV double name(double a, double b) { double r; asm volatile(ptx " %0, %1, %2;" : "=d"(r) : "d"(a), "d"(b)); return r; }
#define IA_VOP3(name, ptx) \
  static IA_DEV double name(double a, double b, double c) { double r; asm volatile(ptx " %0, %1, %2, %3;" : "=d"(r) : "d"(a), "d"(b), "d"(c)); return r; }
  IA_VOP2(add_dn, "add.rm.f64") IA_VOP2(add_up, "add.rp.f64") IA_VOP2(mul_dn, "mul.rm.f64") IA_VOP2(mul_up, "mul.rp.f64")
  IA_VOP2(mul_rn, "mul.rn.f64") IA_VOP3(fma_dn, "fma.rm.f64") IA_VOP3(fma_up, "fma.rp.f64") IA_VOP3(fma_rn, "fma.rn.f64")
#undef IA_VOP2
#undef IA_VOP3
  static IA_DEV double rsqrt_seed(double x) { double y; asm volatile("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x)); return y; }
};
template <> struct VR<float> {
#define IA_VOP2(name, ptx) \
  static IA_DEV float name(float a, float b) { float r; asm volatile(ptx " %0, %1, %2;" : "=f"(r) : "f"(a), "f"(b)); return r; }
#define IA_VOP3(name, ptx) \
  static IA_DEV float name(float a, float b, float c) { float r; asm volatile(ptx " %0, %1, %2, %3;" : "=f"(r) : "f"(a), "f"(b), "f"(c)); return r; }
  IA_VOP2(add_dn, "add.rm.f32") IA_VOP2(add_up, "add.rp.f32") IA_VOP2(mul_dn, "mul.rm.f32") IA_VOP2(mul_up, "mul.rp.f32")
  IA_VOP2(mul_rn, "mul.rn.f32") IA_VOP3(fma_dn, "fma.rm.f32") IA_VOP3(fma_up, "fma.rp.f32") IA_VOP3(fma_rn, "fma.rn.f32")
#undef IA_VOP2
#undef IA_VOP3
};

// ---- quads: one operation on the intervals of both drift signs --------------------------------------
// kinds of "base (+/-) a x" with a in midpoint-radius form
enum { QK_ADD_P = 1, QK_SUB_P = -1, QK_ADD_U = 2, QK_SUB_U = -2 };
template <int SS> struct QKind {            // base + a x / base - a x for a of class SS (a <= 0 is passed negated)
  static constexpr int add = SS > 0 ? QK_ADD_P : (SS < 0 ? QK_SUB_P : QK_ADD_U);
  static constexpr int sub = SS > 0 ? QK_SUB_P : (SS < 0 ? QK_ADD_P : QK_SUB_U);
};
// a as handed to the quad: negated for the class a <= 0
template <int SS, class T> IA_DEV MR<T> q_arg(MR<T> a) { return SS < 0 ? mr_neg(a) : a; }

template <int K, class T>
IA_DEV void q_fma(MR<T> a0, MR<T> a1, Iv<T> x0, Iv<T> x1, Iv<T> b0, Iv<T> b1, Iv<T>& o0, Iv<T>& o1) {
  using V = VR<T>;
  if (K == QK_ADD_P) {
    const T l0 = V::fma_dn(a0.m, x0.lo, b0.lo), h0 = V::fma_up(a0.m, x0.hi, b0.hi);
    const T l1 = V::fma_dn(a1.m, x1.lo, b1.lo), h1 = V::fma_up(a1.m, x1.hi, b1.hi);
    o0.lo = V::fma_dn(-a0.r, fabs(x0.lo), l0); o0.hi = V::fma_up(a0.r, fabs(x0.hi), h0);
    o1.lo = V::fma_dn(-a1.r, fabs(x1.lo), l1); o1.hi = V::fma_up(a1.r, fabs(x1.hi), h1);
  } else if (K == QK_SUB_P) {
    const T l0 = V::fma_dn(-a0.m, x0.hi, b0.lo), h0 = V::fma_up(-a0.m, x0.lo, b0.hi);
    const T l1 = V::fma_dn(-a1.m, x1.hi, b1.lo), h1 = V::fma_up(-a1.m, x1.lo, b1.hi);
    o0.lo = V::fma_dn(-a0.r, fabs(x0.hi), l0); o0.hi = V::fma_up(a0.r, fabs(x0.lo), h0);
    o1.lo = V::fma_dn(-a1.r, fabs(x1.hi), l1); o1.hi = V::fma_up(a1.r, fabs(x1.lo), h1);
  } else {
    if (K == QK_SUB_U) { a0 = mr_neg(a0); a1 = mr_neg(a1); }
    const T p0 = V::fma_dn(a0.m, x0.lo, b0.lo), q0 = V::fma_dn(a0.m, x0.hi, b0.lo);
    const T p1 = V::fma_dn(a1.m, x1.lo, b1.lo), q1 = V::fma_dn(a1.m, x1.hi, b1.lo);
    const T u0 = V::fma_up(a0.m, x0.lo, b0.hi), v0 = V::fma_up(a0.m, x0.hi, b0.hi);
    const T u1 = V::fma_up(a1.m, x1.lo, b1.hi), v1 = V::fma_up(a1.m, x1.hi, b1.hi);
    const T pp0 = V::fma_dn(-a0.r, fabs(x0.lo), p0), qq0 = V::fma_dn(-a0.r, fabs(x0.hi), q0);
    const T pp1 = V::fma_dn(-a1.r, fabs(x1.lo), p1), qq1 = V::fma_dn(-a1.r, fabs(x1.hi), q1);
    const T uu0 = V::fma_up(a0.r, fabs(x0.lo), u0), vv0 = V::fma_up(a0.r, fabs(x0.hi), v0);
    const T uu1 = V::fma_up(a1.r, fabs(x1.lo), u1), vv1 = V::fma_up(a1.r, fabs(x1.hi), v1);
    o0 = {mn(pp0, qq0), mx(uu0, vv0)};
    o1 = {mn(pp1, qq1), mx(uu1, vv1)};
  }
}
// a x for a >= 0 (midpoint-radius)
template <class T> IA_DEV void q_prod_p(MR<T> a, Iv<T> x0, Iv<T> x1, Iv<T>& o0, Iv<T>& o1) {
  using V = VR<T>;
  const T l0 = V::mul_dn(a.m, x0.lo), h0 = V::mul_up(a.m, x0.hi), l1 = V::mul_dn(a.m, x1.lo), h1 = V::mul_up(a.m, x1.hi);
  o0.lo = V::fma_dn(-a.r, fabs(x0.lo), l0); o0.hi = V::fma_up(a.r, fabs(x0.hi), h0);
  o1.lo = V::fma_dn(-a.r, fabs(x1.lo), l1); o1.hi = V::fma_up(a.r, fabs(x1.hi), h1);
}
// c >= 0 per lane times a block-uniform interval s of class SS (SS < 0: s is passed as -s >= 0)
template <int SS, class T> IA_DEV void q_mulpos(Iv<T> c0, Iv<T> c1, Iv<T> s, Iv<T>& o0, Iv<T>& o1) {
  using V = VR<T>;
  if (SS != 0) {
    o0.lo = V::mul_dn(c0.lo, s.lo); o0.hi = V::mul_up(c0.hi, s.hi);
    o1.lo = V::mul_dn(c1.lo, s.lo); o1.hi = V::mul_up(c1.hi, s.hi);
  } else {
    const bool nl = sgn(s.lo), nh = sgn(s.hi);
    o0.lo = V::mul_dn(nl ? c0.hi : c0.lo, s.lo); o0.hi = V::mul_up(nh ? c0.lo : c0.hi, s.hi);
    o1.lo = V::mul_dn(nl ? c1.hi : c1.lo, s.lo); o1.hi = V::mul_up(nh ? c1.lo : c1.hi, s.hi);
  }
}
template <class T> IA_DEV void q_add(Iv<T> a0, Iv<T> a1, Iv<T> b0, Iv<T> b1, Iv<T>& o0, Iv<T>& o1) {
  using V = VR<T>;
  o0.lo = V::add_dn(a0.lo, b0.lo); o0.hi = V::add_up(a0.hi, b0.hi);
  o1.lo = V::add_dn(a1.lo, b1.lo); o1.hi = V::add_up(a1.hi, b1.hi);
}

// largest magnitude among the four endpoints of e (both drift signs), read off the sign-magnitude bit patterns
template <class T> struct EMag;
template <> struct EMag<double> { static constexpr int quarter = 0x3fd00000, sixteenth = 0x3fb00000, one = 0x3ff00000; };
template <> struct EMag<float> { static constexpr int quarter = 0x3e800000, sixteenth = 0x3d800000, one = 0x3f800000; };
template <class T> IA_DEV int e_mag(const Iv<T> (&e)[2]) {
  return max(__vimax3_s32(hiw(e[0].lo) & 0x7fffffff, hiw(e[0].hi) & 0x7fffffff, hiw(e[1].lo) & 0x7fffffff), hiw(e[1].hi) & 0x7fffffff);
}

// sin and cos over e0, e1 inside [-1/4, 1/4] (trig_small of ia_fast.cuh, eight Horner chains abreast)
template <class T> struct TrigC;
template <> struct TrigC<double> {
  static constexpr int NS = 5, NC = 6;
  static IA_DEV double s(int k) { return IA_SIN_C[k]; }
  static IA_DEV double c(int k) { return IA_COS_C[k]; }
  static constexpr int NSM = 9, NCM = 10;            // medium tier (|e| < 1)
  static IA_DEV double sm(int k) { return IA_SIN_M[k]; }
  static IA_DEV double cm(int k) { return IA_COS_M[k]; }
};
template <> struct TrigC<float> {
  static constexpr int NS = 3, NC = 4;
  static IA_DEV float s(int k) { const float c[NS] = {-1.9841270e-04f, 8.3333338e-03f, -1.6666667e-01f}; return c[k]; }
  static IA_DEV float c(int k) { const float d[NC] = {2.4801588e-05f, -1.3888889e-03f, 4.1666668e-02f, -0.5f}; return d[k]; }
  static constexpr int NSM = 5, NCM = 6;
  static IA_DEV float sm(int k) { return Trig<float>::sm(k); }
  static IA_DEV float cm(int k) { return Trig<float>::cm(k); }
};
// short (warp-uniform, double only): every |e| < 2^-4 - the leading coefficients 1/11! (sin) and 1/12!, 1/10! (cos) are
// then below 2^-60 relative (x^10/11! < 2.3e-20; x^10/10! < 2.5e-19 against cos > 0.99) and their three Horner steps
// per point are skipped: 12 FP64 instructions per evaluation.  Same bound as the long form (below 1 ulp, inside the pad).
// medium (warp-uniform): every |e| < 1 - the longer polynomials of ia_fast.cuh (double: terms to x^19 / x^20, float: x^11 / x^12)
template <class T> IA_DEV void q_trig_small(const Iv<T> (&e)[2], Iv<T> (&se)[2], Iv<T> (&ce)[2], bool short_poly = false, bool medium = false) {
  using V = VR<T>;
  using C = TrigC<T>;
  const T x[4] = {e[0].lo, e[0].hi, e[1].lo, e[1].hi};
  T s[4], xs[4], qs[4], qc[4], sn[4], cs[4];
#pragma unroll
  for (int i = 0; i < 4; ++i) s[i] = V::mul_rn(x[i], x[i]);
  if (medium) {
#pragma unroll
    for (int i = 0; i < 4; ++i) { qs[i] = V::fma_rn(C::sm(0), s[i], C::sm(1)); qc[i] = V::fma_rn(C::cm(0), s[i], C::cm(1)); }
#pragma unroll
    for (int k = 2; k < C::NSM; ++k) {
#pragma unroll
      for (int i = 0; i < 4; ++i) { qs[i] = V::fma_rn(qs[i], s[i], C::sm(k)); qc[i] = V::fma_rn(qc[i], s[i], C::cm(k)); }
    }
#pragma unroll
    for (int i = 0; i < 4; ++i) { xs[i] = V::mul_rn(x[i], s[i]); qc[i] = V::fma_rn(qc[i], s[i], C::cm(C::NCM - 1)); }
  } else if (sizeof(T) == 8) {
    // both forms start with an FMA on constants (no register initialisation) and meet after the 1/7! and 1/6! steps
    if (short_poly) {
#pragma unroll
      for (int i = 0; i < 4; ++i) { qs[i] = V::fma_rn(C::s(1), s[i], C::s(2)); qc[i] = V::fma_rn(C::c(2), s[i], C::c(3)); }
    } else {
#pragma unroll
      for (int i = 0; i < 4; ++i) { qs[i] = V::fma_rn(C::s(0), s[i], C::s(1)); qc[i] = V::fma_rn(C::c(0), s[i], C::c(1)); }
#pragma unroll
      for (int i = 0; i < 4; ++i) { qs[i] = V::fma_rn(qs[i], s[i], C::s(2)); qc[i] = V::fma_rn(qc[i], s[i], C::c(2)); }
#pragma unroll
      for (int i = 0; i < 4; ++i) qc[i] = V::fma_rn(qc[i], s[i], C::c(3));
    }
#pragma unroll
    for (int i = 0; i < 4; ++i) xs[i] = V::mul_rn(x[i], s[i]);
#pragma unroll
    for (int i = 0; i < 4; ++i) { qs[i] = V::fma_rn(qs[i], s[i], C::s(3)); qc[i] = V::fma_rn(qc[i], s[i], C::c(4)); }
#pragma unroll
    for (int i = 0; i < 4; ++i) { qs[i] = V::fma_rn(qs[i], s[i], C::s(4)); qc[i] = V::fma_rn(qc[i], s[i], C::c(5)); }
  } else {
#pragma unroll
    for (int i = 0; i < 4; ++i) { qs[i] = V::fma_rn(C::s(0), s[i], C::s(1)); qc[i] = V::fma_rn(C::c(0), s[i], C::c(1)); }
#pragma unroll
    for (int i = 0; i < 4; ++i) xs[i] = V::mul_rn(x[i], s[i]);
#pragma unroll
    for (int k = 2; k < C::NC; ++k) {
#pragma unroll
      for (int i = 0; i < 4; ++i) {
        if (k < C::NS) qs[i] = V::fma_rn(qs[i], s[i], C::s(k));
        qc[i] = V::fma_rn(qc[i], s[i], C::c(k));
      }
    }
  }
#pragma unroll
  for (int i = 0; i < 4; ++i) { sn[i] = V::fma_rn(xs[i], qs[i], x[i]); cs[i] = V::fma_rn(qc[i], s[i], T(1)); }
  T cmin[2], cmax[2];
#pragma unroll
  for (int j = 0; j < 2; ++j) {
    const bool c = nn_gt(s[2 * j], s[2 * j + 1]);
    cmin[j] = c ? cs[2 * j] : cs[2 * j + 1];
    cmax[j] = c ? cs[2 * j + 1] : cs[2 * j];
  }
  T chi[2];
#pragma unroll
  for (int j = 0; j < 2; ++j) {
    se[j].lo = V::fma_dn(-fabs(sn[2 * j]), Rnd<T>::pad_rel(), sn[2 * j]);
    se[j].hi = V::fma_up(fabs(sn[2 * j + 1]), Rnd<T>::pad_rel(), sn[2 * j + 1]);
    ce[j].lo = V::fma_dn(-fabs(cmin[j]), Rnd<T>::pad_rel(), cmin[j]);
    chi[j] = V::fma_up(fabs(cmax[j]), Rnd<T>::pad_rel(), cmax[j]);
  }
#pragma unroll
  for (int j = 0; j < 2; ++j) {
    const bool straddle = sgn(e[j].lo) != sgn(e[j].hi);
    ce[j].hi = (straddle || ge_one(chi[j])) ? T(1) : chi[j];               // cos > 0.96
  }
}

// |delta| = D+ / sqrt(u2) for both signs: four 1/sqrt chains abreast (Dir<double>::rsqrt_near, same bound)
template <class T> struct QDir;
template <> struct QDir<double> {
  static IA_DEV void d_over_sqrt(double DloP, double DhiP, const Iv<double> (&u2)[2], Iv<double> (&dq)[2]) {
    using V = VR<double>;
    const double x[4] = {u2[0].hi, u2[0].lo, u2[1].hi, u2[1].lo};
    double y0[4], t[4], r[4], pp[4], yr[4], y[4];
#pragma unroll
    for (int i = 0; i < 4; ++i) y0[i] = V::rsqrt_seed(x[i]);
#pragma unroll
    for (int i = 0; i < 4; ++i) t[i] = V::mul_rn(x[i], y0[i]);
#pragma unroll
    for (int i = 0; i < 4; ++i) r[i] = V::fma_rn(-t[i], y0[i], 1.0);
#pragma unroll
    for (int i = 0; i < 4; ++i) { pp[i] = V::fma_rn(0.375, r[i], 0.5); yr[i] = V::mul_rn(y0[i], r[i]); }
#pragma unroll
    for (int i = 0; i < 4; ++i) y[i] = V::fma_rn(yr[i], pp[i], y0[i]);
    dq[0].lo = V::mul_dn(DloP, y[0]); dq[0].hi = V::mul_up(DhiP, y[1]);
    dq[1].lo = V::mul_dn(DloP, y[2]); dq[1].hi = V::mul_up(DhiP, y[3]);
  }
};
template <> struct QDir<float> {
  // the same scheme in float: MUFU.RSQ (relative error below 2^-22, PTX rsqrt.approx.f32), one third-order step
  // (result within 2^-23 of 1/sqrt), D+ padded outward by the relative 2^-21 of the float elementary pads.
  // Replaces __fdiv_rd(D, __fsqrt_ru(u2)): two library calls with slow paths per endpoint (4 CALL, 17 BSSY/BSYNC
  // per evaluation in the ncu source page of round 1).
  static IA_DEV void d_over_sqrt(float DloP, float DhiP, const Iv<float> (&u2)[2], Iv<float> (&dq)[2]) {
    using V = VR<float>;
    const float x[4] = {u2[0].hi, u2[0].lo, u2[1].hi, u2[1].lo};
    float y0[4], t[4], r[4], pp[4], yr[4], y[4];
#pragma unroll
    for (int i = 0; i < 4; ++i) asm volatile("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y0[i]) : "f"(x[i]));
#pragma unroll
    for (int i = 0; i < 4; ++i) t[i] = V::mul_rn(x[i], y0[i]);
#pragma unroll
    for (int i = 0; i < 4; ++i) r[i] = V::fma_rn(-t[i], y0[i], 1.0f);
#pragma unroll
    for (int i = 0; i < 4; ++i) { pp[i] = V::fma_rn(0.375f, r[i], 0.5f); yr[i] = V::mul_rn(y0[i], r[i]); }
#pragma unroll
    for (int i = 0; i < 4; ++i) y[i] = V::fma_rn(yr[i], pp[i], y0[i]);
    dq[0].lo = V::mul_dn(DloP, y[0]); dq[0].hi = V::mul_up(DhiP, y[1]);
    dq[1].lo = V::mul_dn(DloP, y[2]); dq[1].hi = V::mul_up(DhiP, y[3]);
  }
};

// ---- two ways to read the per-(block, hit) record inside pass_vote_q ---------------------------------------------
// HitDirect: plain member access (diagnostics, records in local memory).  HitLds: ld.shared from a 32-bit shared-space
// address held in a register - the compiler otherwise rebuilds the record's address in the uniform datapath for every
// group of loads (S2UR SR_CgaCtaId, UMOV, ULEA, UIADD3: 19 instructions per evaluation in the round-2 profile), and an
// instruction that is not an FP64 instruction costs this kernel almost a full issue cycle.  The loads are plain (not
// volatile) asm: the record is read-only after the block's barrier, and the address they depend on is made opaque AFTER
// that barrier (hit_address), so none of them can move above it.
template <class T> struct HitDirect {
  const HitF<T>& r;
  IA_DEV T Tabs() const { return r.Tabs; }
  IA_DEV T DloP() const { return r.DloP; }
  IA_DEV T DhiP() const { return r.DhiP; }
  IA_DEV T band() const { return r.band; }
  IA_DEV int c2cls() const { return r.c2cls; }
  IA_DEV Iv<T> Q() const { return r.Q; }
  IA_DEV Iv<T> cA() const { return r.cA; }
  IA_DEV Iv<T> T2() const { return r.T2; }
  IA_DEV MR<T> cAm() const { return r.cAm; }
  IA_DEV MR<T> iRm() const { return r.iRm; }
  IA_DEV MR<T> TiQm() const { return r.TiQm; }
  IA_DEV MR<T> T2hiQm() const { return r.T2hiQm; }
  IA_DEV MR<T> cA2Tm() const { return r.cA2Tm; }
  IA_DEV Iv<T> sA(int va) const { return r.sA[va]; }
  IA_DEV Iv<T> dphi(int va) const { return r.dphi[va]; }
  IA_DEV Iv<T> sA2(int va) const { return r.sA2[va]; }
  IA_DEV MR<T> sAm(int va) const { return r.sAm[va]; }
  IA_DEV MR<T> s2m(int va) const { return r.s2m[va]; }
};
template <class T> struct LdsOp;
template <> struct LdsOp<double> {
  static IA_DEV void v2(unsigned a, double& x, double& y) { asm("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(x), "=d"(y) : "r"(a)); }
  static IA_DEV double s(unsigned a) { double x; asm("ld.shared.f64 %0, [%1];" : "=d"(x) : "r"(a)); return x; }
};
template <> struct LdsOp<float> {
  static IA_DEV void v2(unsigned a, float& x, float& y) { asm("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(x), "=f"(y) : "r"(a)); }
  static IA_DEV float s(unsigned a) { float x; asm("ld.shared.f32 %0, [%1];" : "=f"(x) : "r"(a)); return x; }
};
#define IA_HOFF(field) unsigned(offsetof(HitF<T>, field))
static_assert(offsetof(HitF<double>, sAm) % 16 == 0 && offsetof(HitF<double>, s2m) % 16 == 0 && offsetof(HitF<double>, sA2) % 16 == 0 &&
              offsetof(HitF<double>, cA2Tm) % 16 == 0 && sizeof(HitF<double>) % 16 == 0, "HitF<double>: pairs must be 16-byte aligned");
static_assert(offsetof(HitF<float>, sAm) % 8 == 0 && offsetof(HitF<float>, s2m) % 8 == 0 && sizeof(HitF<float>) % 16 == 0,
              "HitF<float>: pairs must be 8-byte aligned");
template <class T> struct HitLds {
  unsigned a;            // shared-space address of the record
  IA_DEV Iv<T> iv(unsigned off) const { Iv<T> v; LdsOp<T>::v2(a + off, v.lo, v.hi); return v; }
  IA_DEV MR<T> mr(unsigned off) const { MR<T> v; LdsOp<T>::v2(a + off, v.m, v.r); return v; }
  IA_DEV T Tabs() const { return LdsOp<T>::s(a + IA_HOFF(Tabs)); }
  IA_DEV T DloP() const { return LdsOp<T>::s(a + IA_HOFF(DloP)); }
  IA_DEV T DhiP() const { return LdsOp<T>::s(a + IA_HOFF(DhiP)); }
  IA_DEV T band() const { return LdsOp<T>::s(a + IA_HOFF(band)); }
  IA_DEV int c2cls() const { int x; asm("ld.shared.s32 %0, [%1];" : "=r"(x) : "r"(a + IA_HOFF(c2cls))); return x; }
  IA_DEV Iv<T> Q() const { return iv(IA_HOFF(Q)); }
  IA_DEV Iv<T> cA() const { return iv(IA_HOFF(cA)); }
  IA_DEV Iv<T> T2() const { return iv(IA_HOFF(T2)); }
  IA_DEV MR<T> cAm() const { return mr(IA_HOFF(cAm)); }
  IA_DEV MR<T> iRm() const { return mr(IA_HOFF(iRm)); }
  IA_DEV MR<T> TiQm() const { return mr(IA_HOFF(TiQm)); }
  IA_DEV MR<T> T2hiQm() const { return mr(IA_HOFF(T2hiQm)); }
  IA_DEV MR<T> cA2Tm() const { return mr(IA_HOFF(cA2Tm)); }
  IA_DEV Iv<T> sA(int va) const { return iv(IA_HOFF(sA) + va * unsigned(sizeof(Iv<T>))); }
  IA_DEV Iv<T> dphi(int va) const { return iv(IA_HOFF(dphi) + va * unsigned(sizeof(Iv<T>))); }
  IA_DEV Iv<T> sA2(int va) const { return iv(IA_HOFF(sA2) + va * unsigned(sizeof(Iv<T>))); }
  IA_DEV MR<T> sAm(int va) const { return mr(IA_HOFF(sAm) + va * unsigned(sizeof(MR<T>))); }
  IA_DEV MR<T> s2m(int va) const { return mr(IA_HOFF(s2m) + va * unsigned(sizeof(MR<T>))); }
};
// shared-space address of a record, opaque to the compiler from here on (call after the barrier that publishes the records)
template <class T> IA_DEV unsigned hit_address(const HitF<T>* rec) {
  unsigned a = unsigned(__cvta_generic_to_shared(rec));
  asm volatile("" : "+r"(a));
  return a;
}

// S4-S8 for both drift signs (index 0: D+, 1: D-) of one (cell, hit); returns 1 iff 0 is in f for either.
// Inputs transformed as in ia_fast.cuh: L >= 0, T = h.Tabs >= 0, cA >= 0 (SS != 0) or any (SS == 0).
template <int SS, class T, class H>
IA_DEV unsigned pass_vote_q(const H& h, int va, const Pass2<T>& pc, const PairC<T>& p, const HitP<T>& hp, Iv<T> Zr) {
  // returns decide(): bit 0 the vote, bit 1 (float only) "too close to call in this form"
  using V = VR<T>;
  const T Tn = h.Tabs();
  constexpr int SC = SS == 0 ? 0 : 1;                                  // class of cA inside this body
  const MR<T> sAm = q_arg<SS>(h.sAm(va)), s2m = q_arg<SS>(h.s2m(va));
  // S4: shared part
  Iv<T> zA, t1;
  zA.lo = V::add_dn(Zr.lo, hp.LRdphi.lo); zA.hi = V::add_up(Zr.hi, hp.LRdphi.hi);           // (A.8d)
  {
    const T l = V::mul_dn(p.LRm.m, zA.lo), u = V::mul_up(p.LRm.m, zA.hi);
    t1.lo = V::fma_dn(-p.LRm.r, fabs(zA.lo), l); t1.hi = V::fma_up(p.LRm.r, fabs(zA.hi), u);
  }
  Iv<T> W[2], TY[2], in[2], zG[2], Vv[2], e[2];
  q_fma<QKind<SS>::add>(sAm, sAm, zA, zA, pc.LDcA, ineg(pc.LDcA), W[0], W[1]);              // lambda D cA + zA sA
  if (h.c2cls() == CLS_P) q_fma<QK_SUB_P>(pc.Km[0], pc.Km[1], zA, zA, t1, t1, in[0], in[1]);  // t1 - t2
  else if (h.c2cls() == CLS_N) q_fma<QK_ADD_P>(mr_neg(pc.Km[0]), mr_neg(pc.Km[1]), zA, zA, t1, t1, in[0], in[1]);
  else q_fma<QK_SUB_U>(pc.Km[0], pc.Km[1], zA, zA, t1, t1, in[0], in[1]);
  q_prod_p(h.TiQm(), W[0], W[1], TY[0], TY[1]);                                               // T Phi1 = -TY   (A.8b)
  // G + zA^2: with the pairs of a warp running along R the sign of zA is the same for every lane of most warps - decided
  // per warp: no magnitude sort, no selects (same values: mnn = lo, mag = hi for zA >= 0, the other way round for zA <= 0)
  {
    const bool zpos = __all_sync(0xffffffffu, !sgn(zA.lo)), zneg = __all_sync(0xffffffffu, sgn(zA.hi));
    if (zpos || zneg) {
      const T a = zpos ? zA.lo : zA.hi, b = zpos ? zA.hi : zA.lo;        // smaller, larger magnitude (warp-uniform choice)
      zG[0].lo = V::fma_dn(a, a, pc.G[0].lo); zG[0].hi = V::fma_up(b, b, pc.G[0].hi);
      zG[1].lo = V::fma_dn(a, a, pc.G[1].lo); zG[1].hi = V::fma_up(b, b, pc.G[1].hi);
    } else {
      const Mag<T> gz = mag_of(zA);
      zG[0].lo = V::fma_dn(gz.mnn, gz.mnn, pc.G[0].lo); zG[0].hi = V::fma_up(gz.mag, gz.mag, pc.G[0].hi);
      zG[1].lo = V::fma_dn(gz.mnn, gz.mnn, pc.G[1].lo); zG[1].hi = V::fma_up(gz.mag, gz.mag, pc.G[1].hi);
      if (gz.straddle) { zG[0].lo = pc.G[0].lo; zG[1].lo = pc.G[1].lo; }
    }
  }
  q_fma<QKind<SS>::add>(s2m, s2m, zG[0], zG[1], in[0], in[1], Vv[0], Vv[1]);                // (t1 - t2) + t3
  q_fma<QK_ADD_P>(h.T2hiQm(), h.T2hiQm(), Vv[0], Vv[1], ineg(TY[0]), ineg(TY[1]), e[0], e[1]);  // T^2 Phi2 + T Phi1  (A.8a,c)
  const int emag = e_mag(e);                 // largest |endpoint| of e over both signs, as the high word of the double
  const bool small = emag < EMag<T>::quarter;
  // S5
  Iv<T> se[2], sce[2], cce[2];                                         // sin e, sigma sA cos e, cA cos e
  const bool all_small = __all_sync(0xffffffffu, small);
  if (all_small || __all_sync(0xffffffffu, emag < EMag<T>::one)) {
    Iv<T> ce[2];
    q_trig_small(e, se, ce, all_small && __all_sync(0xffffffffu, emag < EMag<T>::sixteenth), !all_small);
    q_mulpos<SS>(ce[0], ce[1], SS < 0 ? ineg(h.sA(va)) : h.sA(va), sce[0], sce[1]);
    q_mulpos<SC>(ce[0], ce[1], h.cA(), cce[0], cce[1]);
  } else {
    const Trig3<T> g0 = trig_general(e[0], h.sA(va), h.cA()), g1 = trig_general(e[1], h.sA(va), h.cA());
    se[0] = g0.se; cce[0] = g0.cce; sce[0] = SS < 0 ? ineg(g0.sce) : g0.sce;
    se[1] = g1.se; cce[1] = g1.cce; sce[1] = SS < 0 ? ineg(g1.sce) : g1.sce;
  }
  Iv<T> sa[2], ca[2], sinP[2], cosP[2];
  if (SS < 0) q_fma<QKind<SC>::add>(h.cAm(), h.cAm(), se[0], se[1], ineg(sce[0]), ineg(sce[1]), sa[0], sa[1]);
  else q_fma<QKind<SC>::add>(h.cAm(), h.cAm(), se[0], se[1], sce[0], sce[1], sa[0], sa[1]);
  q_fma<QKind<SS>::sub>(sAm, sAm, se[0], se[1], cce[0], cce[1], ca[0], ca[1]);
  q_prod_p(h.iRm(), sa[0], sa[1], sinP[0], sinP[1]);
  q_prod_p(h.iRm(), ca[0], ca[1], cosP[0], cosP[1]);
  // the common case cos Phi >= 0 is decided per warp (cos_nonneg in ia_fast.cuh)
  const bool plain = __all_sync(0xffffffffu, cos_nonneg(cosP));
#pragma unroll
  for (int s = 0; s < 2; ++s) { sinP[s] = clamp_unit(sinP[s]); cosP[s] = clamp_hi(cosP[s]); }
  if (!plain) { cosP[0] = clamp_lo(cosP[0]); cosP[1] = clamp_lo(cosP[1]); }
  // S6: u_d^2 >= 1 - 2 T max|lambda| - rounding >= 0.49 by the guard
  Iv<T> u2[2], dq[2];
  q_fma<QK_ADD_P>(hp.TL2m, hp.TL2m, sinP[0], sinP[1], hp.T2L2, hp.T2L2, u2[0], u2[1]);
  if (plain) {
    const T a0 = V::mul_dn(cosP[0].lo, cosP[0].lo), b0 = V::mul_up(cosP[0].hi, cosP[0].hi);
    const T a1 = V::mul_dn(cosP[1].lo, cosP[1].lo), b1 = V::mul_up(cosP[1].hi, cosP[1].hi);
    u2[0].lo = V::fma_dn(h.T2().lo, a0, u2[0].lo); u2[1].lo = V::fma_dn(h.T2().lo, a1, u2[1].lo);
    u2[0].hi = V::fma_up(h.T2().hi, b0, u2[0].hi); u2[1].hi = V::fma_up(h.T2().hi, b1, u2[1].hi);
  } else {
    const Mag<T> g0 = mag_of(cosP[0]), g1 = mag_of(cosP[1]);
    const T a0 = V::mul_dn(g0.mnn, g0.mnn), b0 = V::mul_up(g0.mag, g0.mag), a1 = V::mul_dn(g1.mnn, g1.mnn), b1 = V::mul_up(g1.mag, g1.mag);
    const T l0 = V::fma_dn(h.T2().lo, a0, u2[0].lo), l1 = V::fma_dn(h.T2().lo, a1, u2[1].lo);
    u2[0].hi = V::fma_up(h.T2().hi, b0, u2[0].hi); u2[1].hi = V::fma_up(h.T2().hi, b1, u2[1].hi);
    u2[0].lo = g0.straddle ? u2[0].lo : l0; u2[1].lo = g1.straddle ? u2[1].lo : l1;
  }
  QDir<T>::d_over_sqrt(h.DloP(), h.DhiP(), u2, dq);                                     // |delta| = D+ / u_d
  // S7: z = (Zr + LR (dphi + e)) - T delta cosP, delta = dq (D+), -dq (D-)
  Iv<T> de[2], zz[2], Tdq[2], TLq[2], qs[2], z[2], ct[2], Rd1[2], Tz[2];
  q_add(e[0], e[1], h.dphi(va), h.dphi(va), de[0], de[1]);
  q_fma<QK_ADD_P>(p.LRm, p.LRm, de[0], de[1], Zr, Zr, zz[0], zz[1]);
  Tdq[0].lo = V::mul_dn(Tn, dq[0].lo); Tdq[0].hi = V::mul_up(Tn, dq[0].hi);                 // |T delta|
  Tdq[1].lo = V::mul_dn(Tn, dq[1].lo); Tdq[1].hi = V::mul_up(Tn, dq[1].hi);
  q_mulpos<1>(Tdq[0], Tdq[1], p.L, TLq[0], TLq[1]);                                         // |T lambda delta|
  q_mulpos<SS>(TLq[0], TLq[1], SS < 0 ? ineg(h.sA2(va)) : h.sA2(va), qs[0], qs[1]);         // sigma 2T |lambda delta| sA
  if (plain) {                                                           // cos Phi >= 0: the partner of .lo is .lo, of .hi is .hi
    z[0].lo = V::fma_dn(-Tdq[0].hi, cosP[0].hi, zz[0].lo); z[0].hi = V::fma_up(-Tdq[0].lo, cosP[0].lo, zz[0].hi);
    z[1].lo = V::fma_dn(Tdq[1].lo, cosP[1].lo, zz[1].lo); z[1].hi = V::fma_up(Tdq[1].hi, cosP[1].hi, zz[1].hi);
  } else {
    const T pl0 = sgn(cosP[0].lo) ? Tdq[0].hi : Tdq[0].lo, ph0 = sgn(cosP[0].hi) ? Tdq[0].lo : Tdq[0].hi;   // partners of cosP.lo / .hi
    const T pl1 = sgn(cosP[1].lo) ? Tdq[1].hi : Tdq[1].lo, ph1 = sgn(cosP[1].hi) ? Tdq[1].lo : Tdq[1].hi;
    z[0].lo = V::fma_dn(-ph0, cosP[0].hi, zz[0].lo); z[0].hi = V::fma_up(-pl0, cosP[0].lo, zz[0].hi);
    z[1].lo = V::fma_dn(pl1, cosP[1].lo, zz[1].lo); z[1].hi = V::fma_up(ph1, cosP[1].hi, zz[1].hi);
  }
  // ct = 2T c^tau (A.7b):  D+: 2T cA z - sigma qs,  D-: 2T cA z + sigma qs
  if (SS < 0) q_fma<QKind<SC>::add>(h.cA2Tm(), h.cA2Tm(), z[0], z[1], qs[0], ineg(qs[1]), ct[0], ct[1]);
  else q_fma<QKind<SC>::add>(h.cA2Tm(), h.cA2Tm(), z[0], z[1], ineg(qs[0]), qs[1], ct[0], ct[1]);
  Rd1[0].lo = V::add_dn(p.R.lo, dq[0].lo); Rd1[0].hi = V::add_up(p.R.hi, dq[0].hi);
  Rd1[1].lo = V::add_dn(p.R.lo, -dq[1].hi); Rd1[1].hi = V::add_up(p.R.hi, -dq[1].lo);
  Tz[0].lo = V::mul_dn(Tn, z[0].lo); Tz[0].hi = V::mul_up(Tn, z[0].hi);
  Tz[1].lo = V::mul_dn(Tn, z[1].lo); Tz[1].hi = V::mul_up(Tn, z[1].hi);
  // S8
  Iv<T> r1[2], r2[2], f[2];
#pragma unroll
  for (int s = 0; s < 2; ++s) { r1[s].lo = V::fma_dn(Rd1[s].lo, Rd1[s].lo, -ct[s].hi); r1[s].hi = V::fma_up(Rd1[s].hi, Rd1[s].hi, -ct[s].lo); }
  {
    const bool tpos = __all_sync(0xffffffffu, (hiw(Tz[0].lo) | hiw(Tz[1].lo)) >= 0);      // z >= 0 for both signs, every lane
    const bool tneg = __all_sync(0xffffffffu, (hiw(Tz[0].hi) & hiw(Tz[1].hi)) < 0);       // z <= 0
    if (tpos || tneg) {
      const T a0 = tpos ? Tz[0].lo : Tz[0].hi, b0 = tpos ? Tz[0].hi : Tz[0].lo;
      const T a1 = tpos ? Tz[1].lo : Tz[1].hi, b1 = tpos ? Tz[1].hi : Tz[1].lo;
      r2[0].lo = V::fma_dn(-b0, b0, r1[0].lo); r2[1].lo = V::fma_dn(-b1, b1, r1[1].lo);
      r2[0].hi = V::fma_up(-a0, a0, r1[0].hi); r2[1].hi = V::fma_up(-a1, a1, r1[1].hi);
    } else {
      const Mag<T> g0 = mag_of(Tz[0]), g1 = mag_of(Tz[1]);
      r2[0].lo = V::fma_dn(-g0.mag, g0.mag, r1[0].lo); r2[1].lo = V::fma_dn(-g1.mag, g1.mag, r1[1].lo);
      const T h0 = V::fma_up(-g0.mnn, g0.mnn, r1[0].hi), h1 = V::fma_up(-g1.mnn, g1.mnn, r1[1].hi);
      r2[0].hi = g0.straddle ? r1[0].hi : h0; r2[1].hi = g1.straddle ? r1[1].hi : h1;
    }
  }
#pragma unroll
  for (int s = 0; s < 2; ++s) { r2[s].lo = V::fma_dn(-TLq[s].hi, TLq[s].hi, r2[s].lo); r2[s].hi = V::fma_up(-TLq[s].lo, TLq[s].lo, r2[s].hi); }
#pragma unroll
  for (int s = 0; s < 2; ++s) { f[s].lo = V::add_dn(h.Q().lo, -r2[s].hi); f[s].hi = V::add_up(h.Q().hi, -r2[s].lo); }
  // inputs are finite and u_d^2 >= 0.49, so f is never NaN here; f.hi is a round-up sum, never -0
  return decide(f, h.band());
}

// ---- one body for all three sign classes ----------------------------------------------------------
// pass_vote_q<SS> compiled three times is 2,750 SASS instructions = 44 KB of hot code; the L1.5
// instruction cache of an SM holds 32 KB.  On fine grids one or two classes dominate and it (just)
// fits; on the coarse 8^5 start grid of a refinement all three classes are live on every SM and the
// kernel starves on instruction fetch (measured on C3: icc hit rate 67 %, stall no_instruction 4.5
// per issue, FP64 pipe 41 %; profiles/r01_c3_ncu.md).  Here the class is a run-time, warp-uniform
// value: the steps that do not depend on it (two thirds of the body) exist once, the five class-
// dependent quads are short uniform switches.  Same arithmetic as pass_vote_q<SS> for every class.
IA_DEV int opaque_i(int x) { asm volatile("" : "+r"(x)); return x; }

// ---- rigorous Phi in the sign-specialised form (ia_params.IA_FLAG_RIGOROUS_PHI; reading f3) ------------------
// atan on [-1/16, 1/16]: odd Taylor polynomial, round-to-nearest Horner; truncation t^14/15 < 2^-59 relative (double,
// terms to t^13) resp. t^8/9 < 2^-35 (float, terms to t^7), rounding below 1 ulp: inside the relative pad 2^-50 (2^-21).
template <class T> struct AtanC;
template <> struct AtanC<double> {
  static IA_DEV double poly(double t) {
    const double s = __dmul_rn(t, t);
    double q = 1.0 / 13.0;
    q = __fma_rn(q, s, -1.0 / 11.0);
    q = __fma_rn(q, s, 1.0 / 9.0);
    q = __fma_rn(q, s, -1.0 / 7.0);
    q = __fma_rn(q, s, 1.0 / 5.0);
    q = __fma_rn(q, s, -1.0 / 3.0);
    return __fma_rn(__dmul_rn(t, s), q, t);
  }
  static constexpr int p4 = 0x3fb00000;            // high word of 2^-4
  static __device__ __noinline__ double lib(double t) { return atan(t); }
  static IA_DEV double rcp(double x) {                 // x in [2^-500, 2^500]; relative error below 2^-51
    double y;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    double e = __fma_rn(-x, y, 1.0);
    y = __fma_rn(y, e, y);
    e = __fma_rn(-x, y, 1.0);
    return __fma_rn(y, e, y);
  }
};
template <> struct AtanC<float> {
  static IA_DEV float poly(float t) {
    const float s = __fmul_rn(t, t);
    float q = -1.0f / 7.0f;
    q = __fmaf_rn(q, s, 1.0f / 5.0f);
    q = __fmaf_rn(q, s, -1.0f / 3.0f);
    return __fmaf_rn(__fmul_rn(t, s), q, t);
  }
  static constexpr int p4 = 0x3d800000;
  static __device__ __noinline__ float lib(float t) { return atanf(t); }
  static IA_DEV float rcp(float x) { return __frcp_rn(x); }
};
// g(E) = atan2(y, x) of the angular equation (A.6) over the rectangle y x x with x > 0: y/x increases with y, and with
// x it decreases where y > 0 and increases where y < 0, so the extremes are at two corners.  ok = false: x may touch 0 -
// the caller re-takes the whole evaluation in the general form (there atan2 on such a rectangle is [-pi, pi]).
template <class T> IA_DEV Iv<T> atan2_small(Iv<T> y, Iv<T> x, bool& ok) {
  using R = Rnd<T>;
  ok = is_pos(x.lo);
  const T xl = ok ? x.lo : T(1), xh = ok ? x.hi : T(1);
  // 1/x in [rl, rh]: a reciprocal good to a few ulps (MUFU seed + two Newton steps, resp. the float instruction), pushed
  // outward by the relative pad - no directed-division subroutine in the loop
  const T rl = pad_dn(AtanC<T>::rcp(xh)), rh = pad_up(AtanC<T>::rcp(xl));
  const T tl = R::mul_dn(y.lo, sgn(y.lo) ? rh : rl), th = R::mul_up(y.hi, sgn(y.hi) ? rl : rh);
  // beyond 1/16 (wide cells): the library's atan, documented maximum error 2 ulp, under the same relative pad
  const bool in = (hiw(tl) & 0x7fffffff) < AtanC<T>::p4 && (hiw(th) & 0x7fffffff) < AtanC<T>::p4;
  T al, ah;
  if (in) { al = AtanC<T>::poly(tl); ah = AtanC<T>::poly(th); }
  else { al = AtanC<T>::lib(tl); ah = AtanC<T>::lib(th); }
  return {pad_dn(al), pad_up(ah)};
}

template <bool RIG = false, class T, class H>
IA_DEV unsigned pass_vote_qr(const H& h, int ss_in, int va, const Pass2<T>& pc, const PairC<T>& p, const HitP<T>& hp,
                             Iv<T> Zr, MR<T> sAm, MR<T> s2m, Iv<T> sAabs, Iv<T> sA2abs, Iv<T>* fout = nullptr) {
  using V = VR<T>;
  const T Tn = h.Tabs();
  // sAm, s2m: negated for the class s_Ax <= 0; sAabs, sA2abs: s_Ax and 2 s_Ax, negated for that class
  const int ss = opaque_i(ss_in);            // keeps the compiler from cloning the loop per class
  // S4: shared part
  Iv<T> zA, t1;
  zA.lo = V::add_dn(Zr.lo, hp.LRdphi.lo); zA.hi = V::add_up(Zr.hi, hp.LRdphi.hi);           // (A.8d)
  {
    const T l = V::mul_dn(p.LRm.m, zA.lo), u = V::mul_up(p.LRm.m, zA.hi);
    t1.lo = V::fma_dn(-p.LRm.r, fabs(zA.lo), l); t1.hi = V::fma_up(p.LRm.r, fabs(zA.hi), u);
  }
  const Mag<T> gz = mag_of(zA);
  Iv<T> W[2], TY[2], in[2], zG[2], Vv[2], e[2];
  if (ss > 0) q_fma<QK_ADD_P>(sAm, sAm, zA, zA, pc.LDcA, ineg(pc.LDcA), W[0], W[1]);        // lambda D cA + zA sA
  else if (ss < 0) q_fma<QK_SUB_P>(sAm, sAm, zA, zA, pc.LDcA, ineg(pc.LDcA), W[0], W[1]);
  else q_fma<QK_ADD_U>(sAm, sAm, zA, zA, pc.LDcA, ineg(pc.LDcA), W[0], W[1]);
  if (h.c2cls() == CLS_P) q_fma<QK_SUB_P>(pc.Km[0], pc.Km[1], zA, zA, t1, t1, in[0], in[1]);  // t1 - t2
  else if (h.c2cls() == CLS_N) q_fma<QK_ADD_P>(mr_neg(pc.Km[0]), mr_neg(pc.Km[1]), zA, zA, t1, t1, in[0], in[1]);
  else q_fma<QK_SUB_U>(pc.Km[0], pc.Km[1], zA, zA, t1, t1, in[0], in[1]);
  q_prod_p(h.TiQm(), W[0], W[1], TY[0], TY[1]);                                               // T Phi1 = -TY   (A.8b)
  zG[0].lo = V::fma_dn(gz.mnn, gz.mnn, pc.G[0].lo); zG[0].hi = V::fma_up(gz.mag, gz.mag, pc.G[0].hi);
  zG[1].lo = V::fma_dn(gz.mnn, gz.mnn, pc.G[1].lo); zG[1].hi = V::fma_up(gz.mag, gz.mag, pc.G[1].hi);
  if (gz.straddle) { zG[0].lo = pc.G[0].lo; zG[1].lo = pc.G[1].lo; }
  if (ss > 0) q_fma<QK_ADD_P>(s2m, s2m, zG[0], zG[1], in[0], in[1], Vv[0], Vv[1]);          // (t1 - t2) + t3
  else if (ss < 0) q_fma<QK_SUB_P>(s2m, s2m, zG[0], zG[1], in[0], in[1], Vv[0], Vv[1]);
  else q_fma<QK_ADD_U>(s2m, s2m, zG[0], zG[1], in[0], in[1], Vv[0], Vv[1]);
  q_fma<QK_ADD_P>(h.T2hiQm(), h.T2hiQm(), Vv[0], Vv[1], ineg(TY[0]), ineg(TY[1]), e[0], e[1]);  // T^2 Phi2 + T Phi1  (A.8a,c)
  // RIG: e is not the series value but a verified enclosure of the fixed point of the angular equation (A.6), obtained by
  // inflation from the series enclosure exactly as in residual_general (ia_residual.cuh; state 0 = verifying, 1 = tightening,
  // 2 = final, per drift sign and lane); S5-S7 below then run once per round for the whole warp.  bad: x of (A.6) is not
  // positive on this lane's box (the wire point may lie on the circle's centre) - the caller re-takes it in the general form.
  int st0 = RIG ? 0 : 2, st1 = RIG ? 0 : 2, rounds0 = 0, rounds1 = 0;
  bool fail0 = false, fail1 = false, bad = false;
  Iv<T> se[2], sce[2], cce[2];                                         // sin e, sigma sA cos e, cA cos e
  Iv<T> sa[2], ca[2], sinP[2], cosP[2];
  Iv<T> u2[2], dq[2];
  Iv<T> de[2], zz[2], Tdq[2], TLq[2], qs[2], z[2], ct[2], Rd1[2], Tz[2];
#pragma unroll 1
  for (;;) {
  const int emag = e_mag(e);                 // largest |endpoint| of e over both signs, as the high word of the double
  const bool small = emag < EMag<T>::quarter;
  // S5
  const bool all_small = __all_sync(0xffffffffu, small);
  if (all_small || __all_sync(0xffffffffu, emag < EMag<T>::one)) {
    Iv<T> ce[2];
    q_trig_small(e, se, ce, all_small && __all_sync(0xffffffffu, emag < EMag<T>::sixteenth), !all_small);
    if (ss != 0) {
      q_mulpos<1>(ce[0], ce[1], sAabs, sce[0], sce[1]);
      q_mulpos<1>(ce[0], ce[1], h.cA(), cce[0], cce[1]);
    } else {
      q_mulpos<0>(ce[0], ce[1], sAabs, sce[0], sce[1]);
      q_mulpos<0>(ce[0], ce[1], h.cA(), cce[0], cce[1]);
    }
  } else {
    const Trig3<T> g0 = trig_general(e[0], h.sA(va), h.cA()), g1 = trig_general(e[1], h.sA(va), h.cA());
    se[0] = g0.se; cce[0] = g0.cce; sce[0] = ss < 0 ? ineg(g0.sce) : g0.sce;
    se[1] = g1.se; cce[1] = g1.cce; sce[1] = ss < 0 ? ineg(g1.sce) : g1.sce;
  }
  if (ss > 0) {
    q_fma<QK_ADD_P>(h.cAm(), h.cAm(), se[0], se[1], sce[0], sce[1], sa[0], sa[1]);
    q_fma<QK_SUB_P>(sAm, sAm, se[0], se[1], cce[0], cce[1], ca[0], ca[1]);
  } else if (ss < 0) {
    q_fma<QK_ADD_P>(h.cAm(), h.cAm(), se[0], se[1], ineg(sce[0]), ineg(sce[1]), sa[0], sa[1]);
    q_fma<QK_ADD_P>(sAm, sAm, se[0], se[1], cce[0], cce[1], ca[0], ca[1]);
  } else {
    q_fma<QK_ADD_U>(h.cAm(), h.cAm(), se[0], se[1], sce[0], sce[1], sa[0], sa[1]);
    q_fma<QK_SUB_U>(sAm, sAm, se[0], se[1], cce[0], cce[1], ca[0], ca[1]);
  }
  q_prod_p(h.iRm(), sa[0], sa[1], sinP[0], sinP[1]);
  q_prod_p(h.iRm(), ca[0], ca[1], cosP[0], cosP[1]);
  // the common case cos Phi >= 0 is decided per warp (cos_nonneg in ia_fast.cuh)
  const bool plain = __all_sync(0xffffffffu, cos_nonneg(cosP));
#pragma unroll
  for (int s = 0; s < 2; ++s) { sinP[s] = clamp_unit(sinP[s]); cosP[s] = clamp_hi(cosP[s]); }
  if (!plain) { cosP[0] = clamp_lo(cosP[0]); cosP[1] = clamp_lo(cosP[1]); }
  // S6: u_d^2 >= 1 - 2 T max|lambda| - rounding >= 0.49 by the guard
  q_fma<QK_ADD_P>(hp.TL2m, hp.TL2m, sinP[0], sinP[1], hp.T2L2, hp.T2L2, u2[0], u2[1]);
  if (plain) {
    const T a0 = V::mul_dn(cosP[0].lo, cosP[0].lo), b0 = V::mul_up(cosP[0].hi, cosP[0].hi);
    const T a1 = V::mul_dn(cosP[1].lo, cosP[1].lo), b1 = V::mul_up(cosP[1].hi, cosP[1].hi);
    u2[0].lo = V::fma_dn(h.T2().lo, a0, u2[0].lo); u2[1].lo = V::fma_dn(h.T2().lo, a1, u2[1].lo);
    u2[0].hi = V::fma_up(h.T2().hi, b0, u2[0].hi); u2[1].hi = V::fma_up(h.T2().hi, b1, u2[1].hi);
  } else {
    const Mag<T> g0 = mag_of(cosP[0]), g1 = mag_of(cosP[1]);
    const T a0 = V::mul_dn(g0.mnn, g0.mnn), b0 = V::mul_up(g0.mag, g0.mag), a1 = V::mul_dn(g1.mnn, g1.mnn), b1 = V::mul_up(g1.mag, g1.mag);
    const T l0 = V::fma_dn(h.T2().lo, a0, u2[0].lo), l1 = V::fma_dn(h.T2().lo, a1, u2[1].lo);
    u2[0].hi = V::fma_up(h.T2().hi, b0, u2[0].hi); u2[1].hi = V::fma_up(h.T2().hi, b1, u2[1].hi);
    u2[0].lo = g0.straddle ? u2[0].lo : l0; u2[1].lo = g1.straddle ? u2[1].lo : l1;
  }
  QDir<T>::d_over_sqrt(h.DloP(), h.DhiP(), u2, dq);                                     // |delta| = D+ / u_d
  // S7: z = (Zr + LR (dphi + e)) - T delta cosP, delta = dq (D+), -dq (D-)
  q_add(e[0], e[1], h.dphi(va), h.dphi(va), de[0], de[1]);
  q_fma<QK_ADD_P>(p.LRm, p.LRm, de[0], de[1], Zr, Zr, zz[0], zz[1]);
  Tdq[0].lo = V::mul_dn(Tn, dq[0].lo); Tdq[0].hi = V::mul_up(Tn, dq[0].hi);                 // |T delta|
  Tdq[1].lo = V::mul_dn(Tn, dq[1].lo); Tdq[1].hi = V::mul_up(Tn, dq[1].hi);
  q_mulpos<1>(Tdq[0], Tdq[1], p.L, TLq[0], TLq[1]);                                         // |T lambda delta|
  if (plain) {                                                           // cos Phi >= 0: the partner of .lo is .lo, of .hi is .hi
    z[0].lo = V::fma_dn(-Tdq[0].hi, cosP[0].hi, zz[0].lo); z[0].hi = V::fma_up(-Tdq[0].lo, cosP[0].lo, zz[0].hi);
    z[1].lo = V::fma_dn(Tdq[1].lo, cosP[1].lo, zz[1].lo); z[1].hi = V::fma_up(Tdq[1].hi, cosP[1].hi, zz[1].hi);
  } else {
    const T pl0 = sgn(cosP[0].lo) ? Tdq[0].hi : Tdq[0].lo, ph0 = sgn(cosP[0].hi) ? Tdq[0].lo : Tdq[0].hi;   // partners of cosP.lo / .hi
    const T pl1 = sgn(cosP[1].lo) ? Tdq[1].hi : Tdq[1].lo, ph1 = sgn(cosP[1].hi) ? Tdq[1].lo : Tdq[1].hi;
    z[0].lo = V::fma_dn(-ph0, cosP[0].hi, zz[0].lo); z[0].hi = V::fma_up(-pl0, cosP[0].lo, zz[0].hi);
    z[1].lo = V::fma_dn(pl1, cosP[1].lo, zz[1].lo); z[1].hi = V::fma_up(ph1, cosP[1].hi, zz[1].hi);
  }
  // qs = sigma 2T |lambda delta| sA;  ct = 2T c^tau (A.7b):  D+: 2T cA z - sigma qs,  D-: 2T cA z + sigma qs
  if (ss > 0) {
    q_mulpos<1>(TLq[0], TLq[1], sA2abs, qs[0], qs[1]);
    q_fma<QK_ADD_P>(h.cA2Tm(), h.cA2Tm(), z[0], z[1], ineg(qs[0]), qs[1], ct[0], ct[1]);
  } else if (ss < 0) {
    q_mulpos<1>(TLq[0], TLq[1], sA2abs, qs[0], qs[1]);
    q_fma<QK_ADD_P>(h.cA2Tm(), h.cA2Tm(), z[0], z[1], qs[0], ineg(qs[1]), ct[0], ct[1]);
  } else {
    q_mulpos<0>(TLq[0], TLq[1], sA2abs, qs[0], qs[1]);
    q_fma<QK_ADD_U>(h.cA2Tm(), h.cA2Tm(), z[0], z[1], ineg(qs[0]), qs[1], ct[0], ct[1]);
  }
  Rd1[0].lo = V::add_dn(p.R.lo, dq[0].lo); Rd1[0].hi = V::add_up(p.R.hi, dq[0].hi);
  Rd1[1].lo = V::add_dn(p.R.lo, -dq[1].hi); Rd1[1].hi = V::add_up(p.R.hi, -dq[1].lo);
  Tz[0].lo = V::mul_dn(Tn, z[0].lo); Tz[0].hi = V::mul_up(Tn, z[0].hi);
  Tz[1].lo = V::mul_dn(Tn, z[1].lo); Tz[1].hi = V::mul_up(Tn, z[1].hi);
  if (!RIG) break;
  if (__all_sync(0xffffffffu, (st0 == 2 || fail0 || bad) && (st1 == 2 || fail1 || bad))) break;
  {
    // g(E) = atan2(T s^tau, R_Ax^2 + T c^tau), s^tau = -(z s_Ax + lambda delta c_Ax) (A.6), (A.7b,c); here T z = Tz,
    // T lambda delta = +-TLq (D+ / D-), 2 T c^tau = ct
    using Rd = Rnd<T>;
    const T tiny = sizeof(T) == 4 ? T(1e-6) : T(1e-12);
    const MR<T> sAt = h.sAm(va), cAt = h.cAm();          // true signs (universal products: any class)
#pragma unroll
    for (int s = 0; s < 2; ++s) {
      const Iv<T> zs = prod_u(sAt, Tz[s]), lc = prod_u(cAt, TLq[s]);
      const Iv<T> sum = s == 0 ? iadd(zs, lc) : isub(zs, lc);
      const Iv<T> y = ineg(sum);
      const Iv<T> x = {Rd::add_dn(h.Q().lo, Rd::mul_dn(T(0.5), ct[s].lo)), Rd::add_up(h.Q().hi, Rd::mul_up(T(0.5), ct[s].hi))};
      bool ok;
      const Iv<T> G = atan2_small(y, x, ok);
      int& st = s == 0 ? st0 : st1;
      int& rounds = s == 0 ? rounds0 : rounds1;
      bool& fail = s == 0 ? fail0 : fail1;
      if (!ok) bad = true;
      if (st == 0) {
        if (G.lo >= e[s].lo && G.hi <= e[s].hi) {
          e[s] = G;
          st = 1;
        } else {
          if (++rounds >= 6) { fail = true; st = 2; }
          const T lo_h = mn(e[s].lo, G.lo), hi_h = mx(e[s].hi, G.hi);
          const T pad = Rd::add_up(Rd::mul_up(T(0.1), Rd::add_up(hi_h, -lo_h)), tiny);
          e[s] = {Rd::add_dn(lo_h, -pad), Rd::add_up(hi_h, pad)};
        }
      } else if (st == 1) {
        e[s] = {mx(e[s].lo, G.lo), mn(e[s].hi, G.hi)};
        if (!(e[s].lo <= e[s].hi)) { fail = true; e[s] = G; }
        st = 2;
      }
    }
    if (bad) { e[0] = e[1] = Iv<T>{T(0), T(0)}; }
  }
  }
  // S8
  Iv<T> r1[2], r2[2], f[2];
#pragma unroll
  for (int s = 0; s < 2; ++s) { r1[s].lo = V::fma_dn(Rd1[s].lo, Rd1[s].lo, -ct[s].hi); r1[s].hi = V::fma_up(Rd1[s].hi, Rd1[s].hi, -ct[s].lo); }
  {
    const Mag<T> g0 = mag_of(Tz[0]), g1 = mag_of(Tz[1]);
    r2[0].lo = V::fma_dn(-g0.mag, g0.mag, r1[0].lo); r2[1].lo = V::fma_dn(-g1.mag, g1.mag, r1[1].lo);
    const T h0 = V::fma_up(-g0.mnn, g0.mnn, r1[0].hi), h1 = V::fma_up(-g1.mnn, g1.mnn, r1[1].hi);
    r2[0].hi = g0.straddle ? r1[0].hi : h0; r2[1].hi = g1.straddle ? r1[1].hi : h1;
  }
#pragma unroll
  for (int s = 0; s < 2; ++s) { r2[s].lo = V::fma_dn(-TLq[s].hi, TLq[s].hi, r2[s].lo); r2[s].hi = V::fma_up(-TLq[s].lo, TLq[s].lo, r2[s].hi); }
#pragma unroll
  for (int s = 0; s < 2; ++s) { f[s].lo = V::add_dn(h.Q().lo, -r2[s].hi); f[s].hi = V::add_up(h.Q().hi, -r2[s].lo); }
  if (fout) { fout[0] = f[0]; fout[1] = f[1]; }       // diagnostics (ia_residual_fast); nullptr in the vote kernels
  unsigned r = decide(f, h.band());
  if (RIG) {
    if (fail0 || fail1) r |= 1u;                      // not verified: the hit votes (cannot exclude), as in the general form
    if (bad) r |= 4u;                                 // outside the fast form's domain: re-take in the general form
  }
  return r;
}

}  // namespace ia
