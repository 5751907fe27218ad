// ia_residual.cuh - the residual enclosure of one (box, hit, drift sign): steps S1-S8 of DESIGN.md.
//
//   f = R_Ax^2 - (R + d_Ax)^2                         eq. (2)/(A.5a)
//   (R + d_Ax)^2 = (R+delta)^2 - 2 c^tau T - (z_St T)^2 - (lambda delta T)^2,  delta = d_St/u_d
//                                                      radicand of (A.5b), L183
//   Phi = Phi_Ax + T Phi1 + T^2 Phi2                  series (A.8a-d), L209-218
// evaluated in interval arithmetic; the hit votes iff 0 is in f for either drift sign, eq. (4) L76.
//
// This header holds the GENERAL form: every product takes the min/max of its four endpoint
// products, nothing is assumed about signs.  It serves the explicit-box kernels, the diagnostics
// and the rare dense tiles whose lambda cells straddle 0; the dense fast path (ia_vote.cu)
// computes the same expression DAG with sign-specialised products.
#pragma once
#include "ia_interval.cuh"

namespace ia {

// per-hit scalars, round-to-nearest, unfused, then taken as exact (S2, S3)
template <class T> struct HitC {
  T xA, yA;          // (A.4d,e) L174-176: wire point in the plane z = z_ref
  T sphi, cphi, Tn;  // sin phi_s, cos phi_s, tan tau
  T k0, kx, ky;      // S3 cross term  k0 + ky*X + kx*Y
  T mx, my, h2;      // S3 dot term    (X-mx)^2 + (Y-my)^2 - h2
  T Dlo, Dhi;        // S1: D+ = [max(d-tol,0), d+tol]
  T zref;
  int valid;         // 0: hit names an unknown wire -> never votes
  int _pad;
};

// the part of HitC the (R, z0, lambda) stage needs
template <class T> struct HitS {
  T Tn, Dlo, Dhi;
  int valid;
  int rig;           // params.IA_FLAG_RIGOROUS_PHI: rigorous enclosure of Phi (reading f3), carried in HitC::_pad
};
template <class T> IA_DEV HitS<T> hit_small(const HitC<T>& c) { return {c.Tn, c.Dlo, c.Dhi, c.valid, c._pad}; }

// what depends on (xc, yc, hit) only: S2, S3, S3'
template <class T> struct XYInv {
  Iv<T> Q, cA, sA, dphi, iQ, RA, iR, c2, s2;
  int forced;        // Q.lo <= 0: the xy cell may contain the wire point -> vote (G15)
};

template <class T> struct Box3 { Iv<T> R, Z, L; };

struct Resid { double flo, fhi, scale; int forced; };

template <class T> IA_DEV XYInv<T> xy_invariants(Iv<T> X, Iv<T> Y, const HitC<T>& c) {
  XYInv<T> v;
  // S2 (A.7a,d,e) L191-201
  Iv<T> A = isub(thin(c.xA), X), B = isub(thin(c.yA), Y);
  v.Q = iadd(isqr(A), isqr(B));
  v.cA = isub(iscale(c.sphi, A), iscale(c.cphi, B));
  v.sA = iadd(iscale(c.cphi, A), iscale(c.sphi, B));
  v.forced = !(v.Q.lo > T(0));
  if (v.forced) {
    v.dphi = v.iQ = v.RA = v.iR = v.c2 = v.s2 = Iv<T>{T(0), T(0)};
    return v;
  }
  // S3 turning angle phi_Ax - phi0, (1d) L49 and (A.7f) L203 as one atan2(cross, dot) (G8)
  Iv<T> cr = iadd(iadd(thin(c.k0), iscale(c.ky, X)), iscale(c.kx, Y));
  Iv<T> dt = isub(iadd(isqr(isub(X, thin(c.mx))), isqr(isub(Y, thin(c.my)))), thin(c.h2));
  v.dphi = iatan2(cr, dt);
  // S3' (A.7a,g): 1/R_Ax^2, R_Ax, 1/R_Ax, cos 2Phi_Ax, sin 2Phi_Ax
  v.iQ = irecip_pos(v.Q);
  v.RA = isqrt(v.Q);
  v.iR = irecip_pos(v.RA);
  v.c2 = imul(isub(isqr(v.cA), isqr(v.sA)), v.iQ);
  v.s2 = imul(iscale(T(2), imul(v.sA, v.cA)), v.iQ);
  return v;
}

// S4-S8 for one drift sign (sign = +1 / -1)
template <class T> IA_DEV Resid residual_general(const Box3<T>& b, const XYInv<T>& v, const HitS<T>& c, T zref, int sign) {
  using Rd = Rnd<T>;
  if (v.forced) return {0.0, 0.0, double(v.Q.hi), 1};
  Iv<T> D = {c.Dlo, c.Dhi};
  if (sign < 0) D = ineg(D);
  const T Tn = c.Tn;
  // S4 (A.8a-d)
  Iv<T> Zr = isub(b.Z, thin(zref));
  Iv<T> LR = imul(b.L, b.R);
  Iv<T> zA = iadd(Zr, imul(LR, v.dphi));                                            // (A.8d)
  Iv<T> LD = imul(b.L, D);
  Iv<T> P1 = ineg(imul(iadd(imul(zA, v.sA), imul(LD, v.cA)), v.iQ));                // (A.8b)
  Iv<T> t1 = imul(LR, zA);
  Iv<T> t2 = imul(imul(imul(b.L, zA), isub(b.R, iscale(T(2), D))), v.c2);
  Iv<T> t3 = imul(iadd(isqr(zA), imul(D, iadd(v.RA, imul(isqr(b.L), isub(iadd(b.R, v.RA), D))))), v.s2);
  Iv<T> P2 = iscale(T(0.5), imul(iadd(isub(t1, t2), t3), v.iQ));                    // (A.8c)
  Iv<T> T2 = isqr(thin(Tn));
  Iv<T> e = iadd(iscale(Tn, P1), imul(T2, P2));                                     // (A.8a)
  // S5-S7 as a function of e = Phi - Phi_Ax: evaluated once with the series value, or - rigorous mode - several
  // times inside the verification of the fixed point of (A.6)
  const T twoT = Rd::mul_rn(T(2), Tn);
  Iv<T> sinP, cosP, dl, z, Ld, ct;
  bool u_ok = true;
  auto s5_to_s7 = [&](Iv<T> ee) {
    // S5 sin/cos of Phi = Phi_Ax + e, (A.3b) and (A.7g)
    Iv<T> se = isin(ee), ce = icos(ee);
    sinP = iclamp(imul(iadd(imul(v.sA, ce), imul(v.cA, se)), v.iR), T(-1), T(1));
    cosP = iclamp(imul(isub(imul(v.cA, ce), imul(v.sA, se)), v.iR), T(-1), T(1));
    // S6 (A.3a) L160 and delta = d_St/u_d
    Iv<T> u2 = iadd(iadd(iadd(thin(T(1)), iscale(twoT, imul(b.L, sinP))), imul(T2, isqr(b.L))), imul(T2, isqr(cosP)));
    Iv<T> u = isqrt(u2);
    if (!(u.lo > T(0))) { u_ok = false; return; }
    dl = idiv_pos(D, u);
    // S7 (A.4c) L172 with s_perp = R (dphi + e);  c^tau of (A.7b) L194
    z = isub(iadd(Zr, imul(LR, iadd(v.dphi, ee))), iscale(Tn, imul(dl, cosP)));
    Ld = imul(b.L, dl);
    ct = isub(imul(z, v.cA), imul(Ld, v.sA));
  };
  // Rigorous mode, reading f3 (PAPER.md L187 eq. (A.6)): e is a fixed point of
  //   g(e) = atan2(T s^tau(e), R_Ax^2 + T c^tau(e)),  s^tau = -z s_Ax - lambda delta c_Ax     (A.6), (A.7b,c)
  // Verification by inflation from the series enclosure: g(E) inside E => a fixed point lies in g(E); then
  // E := g(E), and once more E := g(E) meet E.  Otherwise E := hull(E, g(E)) widened by a tenth of its width
  // (+ a small absolute amount), at most 6 rounds; not verified: the hit votes (cannot exclude).
  // One loop, one copy of S5-S7 in the binary: state 0 = verifying, 1 = tightening, 2 = the evaluation that S8 uses
  // (the series mode enters in state 2).  Three inlined copies per drift sign starved the kernel on instruction
  // fetch (icc hit rate 44 %).
  const T tiny = sizeof(T) == 4 ? T(1e-6) : T(1e-12);
  int state = c.rig ? 0 : 2, rounds = 0;
#pragma unroll 1
  for (;;) {
    s5_to_s7(e);
    if (!u_ok) return {0.0, 0.0, double(v.Q.hi), 1};
    if (state == 2) break;
    const Iv<T> st = ineg(iadd(imul(z, v.sA), imul(Ld, v.cA)));
    const Iv<T> G = iatan2(iscale(Tn, st), iadd(v.Q, iscale(Tn, ct)));
    if (state == 0) {
      if (G.lo >= e.lo && G.hi <= e.hi) {
        e = G;
        state = 1;
      } else {
        if (++rounds >= 6) return {0.0, 0.0, double(v.Q.hi), 1};
        const T lo_h = mn(e.lo, G.lo), hi_h = mx(e.hi, G.hi);
        const T pad = Rd::add_up(Rd::mul_up(T(0.1), Rd::add_up(hi_h, -lo_h)), tiny);
        e = {Rd::add_dn(lo_h, -pad), Rd::add_up(hi_h, pad)};
      }
    } else {
      e = {mx(e.lo, G.lo), mn(e.hi, G.hi)};
      if (!(e.lo <= e.hi)) return {0.0, 0.0, double(v.Q.hi), 1};
      state = 2;
    }
  }
  // S8 radicand of (A.5b) L183 and f of (A.5a) L180
  Iv<T> rad = isub(isub(isub(isqr(iadd(b.R, dl)), iscale(twoT, ct)), isqr(iscale(Tn, z))), isqr(iscale(Tn, Ld)));
  Iv<T> f = isub(v.Q, rad);
  double sc = fmax(double(v.Q.hi), fmax(fabs(double(rad.lo)), fabs(double(rad.hi))));
  return {double(f.lo), double(f.hi), sc, 0};
}

IA_DEV bool resid_votes(const Resid& r) { return r.forced || !(r.flo > 0.0 || r.fhi < 0.0); }

template <class T> IA_DEV bool hit_votes_general(const Box3<T>& b, const XYInv<T>& v, const HitS<T>& c, T zref) {
  if (!c.valid) return false;
  // one copy of the residual in the binary for both drift signs (the general kernels are bound by instruction fetch)
#pragma unroll 1
  for (int s = 0; s < 2; ++s)
    if (resid_votes(residual_general(b, v, c, zref, s == 0 ? +1 : -1))) return true;
  return false;
}

// outward conversion of a double box [lo, hi] to T endpoints (G22)
template <class T> IA_DEV Iv<T> box_iv(double lo, double hi) { return {Rnd<T>::from_dn(lo), Rnd<T>::from_up(hi)}; }

// dense-grid cell edge e_k = lo + k*w, e_n = hi; round-to-nearest, unfused (S9, G14)
IA_DEV double cell_edge(double lo, double hi, double w, int k, int n) {
  return k >= n ? hi : __dadd_rn(lo, __dmul_rn(double(k), w));
}

}  // namespace ia
