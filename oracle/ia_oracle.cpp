// ia_oracle.cpp - the ORACLE.  TEST INFRASTRUCTURE, NOT PRODUCT.
//
// A plain, slow, obviously-correct CPU implementation of the interval-arithmetic helix vote of
// arxiv 2401.04576, written from the paper before any CUDA kernel existed.  It shares
// no code, header, table or constant with the CUDA path under paper_2401_04576_b200/csrc and is
// never called by it.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
// --impl reference leg may load this library.
//
// What it computes (citations are PAPER.md line numbers; "S<n>"/"G<n>" are the step and reading
// numbers of DESIGN.md, which restate SURVEY.md 8(c)):
//   for every 5-D box  (xc, yc, R, z0, lambda)  and every hit (wire, |drift|):
//     the interval extension of the stereo-generalised Apollonius residual, eq. (2)/(A.5a) L55,L180,
//         f = (x_Ax - xc)^2 + (y_Ax - yc)^2 - (R + d_Ax)^2 ,   (R + d_Ax)^2 = radicand of (A.5b) L183
//     with the angle Phi of (A.3b) taken from the second-order series (A.8a-d) L209-218,
//     evaluated for both drift signs; the hit votes for the box iff 0 is in the enclosure for
//     either sign (condition (4), L74-78).  votes[box] = number of hits that vote.
//   top-K by (votes desc, index asc); refinement by 2^5 midpoint subdivision of the top-K boxes.
//
// Rounding: every interval primitive returns the tightest enclosure IEEE-754 allows: lower
// endpoints rounded toward -inf, upper endpoints toward +inf.  The thread keeps the FPU in
// FE_UPWARD while interval code runs and obtains round-down results through the identity
//     RD(x op y) = -RU((-x) op y)            (op in {+, *, /};  x - y = x + (-y))
// sqrt toward -inf switches the mode for that one instruction.  libm calls (sin, cos, atan2) are
// made in FE_TONEAREST and widened by ELEM_PAD_ULPS ulps on each side with nextafter (glibc
// documents <= 1 ulp for these; 4 leaves margin), then clamped to the mathematical range.
// Build flags: -O2 -frounding-math -ffp-contract=off -fno-fast-math -fno-math-errno  (see build.py)
//
// Pins (tests/test_oracle_*.py, all -m "not gpu"):  P1 identity at the generated truth,
// P3 containment, P4 axial closed form, P5 brute-force sampling, P6 inclusion isotonicity,
// P8 series order, P9 independent round-to-nearest DAG anchor; primitives against exact
// rational arithmetic.  Paper mode (orc_vote_paper ...): MP1-MP6; iteration scheme (orc_disk_filter,
// orc_select_max_paper, orc_find_hits_paper, orc_track_paper): F2a-F2e, M6; rigorous Phi (flags bit 4): R1-R3.
// Parity status: pinned (none of the functions here is "parity unpinned").

#include <algorithm>
#include <cfenv>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <limits>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

constexpr int ELEM_PAD_ULPS = 4;

// keep the optimiser from moving or folding a rounded operation
template <class T> inline T opaque(T x) { asm volatile("" : "+x"(x)); return x; }

struct UpMode {       // RAII: FE_UPWARD for the lifetime of the object
  int saved;
  UpMode() : saved(fegetround()) { fesetround(FE_UPWARD); }
  ~UpMode() { fesetround(saved); }
};
struct NearestInUp {  // RAII: FE_TONEAREST inside an UpMode region
  NearestInUp() { fesetround(FE_TONEAREST); }
  ~NearestInUp() { fesetround(FE_UPWARD); }
};

// ---- directed scalar operations (mode must be FE_UPWARD) -------------------------------------
template <class T> inline T up_add(T a, T b) { return opaque(opaque(a) + opaque(b)); }
template <class T> inline T dn_add(T a, T b) { return -opaque(opaque(-a) - opaque(b)); }
template <class T> inline T up_mul(T a, T b) { return opaque(opaque(a) * opaque(b)); }
template <class T> inline T dn_mul(T a, T b) { return -opaque(opaque(-a) * opaque(b)); }
template <class T> inline T up_div(T a, T b) { return opaque(opaque(a) / opaque(b)); }
template <class T> inline T dn_div(T a, T b) { return -opaque(opaque(-a) / opaque(b)); }
template <class T> inline T up_sqrt(T a) { return opaque(std::sqrt(opaque(a))); }
template <class T> inline T dn_sqrt(T a) {
  fesetround(FE_DOWNWARD);
  T r = opaque(std::sqrt(opaque(a)));
  fesetround(FE_UPWARD);
  return r;
}

// ---- intervals ------------------------------------------------------------------------------
template <class T> struct Iv { T lo, hi; };
template <class T> inline Iv<T> thin(T x) { return {x, x}; }

template <class T> inline Iv<T> iadd(Iv<T> a, Iv<T> b) { return {dn_add(a.lo, b.lo), up_add(a.hi, b.hi)}; }
template <class T> inline Iv<T> isub(Iv<T> a, Iv<T> b) { return {dn_add(a.lo, -b.hi), up_add(a.hi, -b.lo)}; }
template <class T> inline Iv<T> ineg(Iv<T> a) { return {-a.hi, -a.lo}; }
template <class T> inline Iv<T> imul(Iv<T> a, Iv<T> b) {
  T l = std::min(std::min(dn_mul(a.lo, b.lo), dn_mul(a.lo, b.hi)), std::min(dn_mul(a.hi, b.lo), dn_mul(a.hi, b.hi)));
  T h = std::max(std::max(up_mul(a.lo, b.lo), up_mul(a.lo, b.hi)), std::max(up_mul(a.hi, b.lo), up_mul(a.hi, b.hi)));
  return {l, h};
}
// exact scalar times interval
template <class T> inline Iv<T> iscale(T c, Iv<T> a) {
  if (c >= 0) return {dn_mul(c, a.lo), up_mul(c, a.hi)};
  return {dn_mul(c, a.hi), up_mul(c, a.lo)};
}
template <class T> inline Iv<T> isqr(Iv<T> a) {
  if (a.lo >= 0) return {dn_mul(a.lo, a.lo), up_mul(a.hi, a.hi)};
  if (a.hi <= 0) return {dn_mul(a.hi, a.hi), up_mul(a.lo, a.lo)};
  return {T(0), std::max(up_mul(a.lo, a.lo), up_mul(a.hi, a.hi))};
}
// a / b with b.lo > 0
template <class T> inline Iv<T> idiv_pos(Iv<T> a, Iv<T> b) {
  T l = a.lo >= 0 ? dn_div(a.lo, b.hi) : dn_div(a.lo, b.lo);
  T h = a.hi >= 0 ? up_div(a.hi, b.lo) : up_div(a.hi, b.hi);
  return {l, h};
}
template <class T> inline Iv<T> irecip_pos(Iv<T> b) { return {dn_div(T(1), b.hi), up_div(T(1), b.lo)}; }
// sqrt of the non-negative part
template <class T> inline Iv<T> isqrt(Iv<T> a) {
  return {dn_sqrt(std::max(a.lo, T(0))), up_sqrt(std::max(a.hi, T(0)))};
}
template <class T> inline Iv<T> iclamp(Iv<T> a, T lo, T hi) { return {std::max(a.lo, lo), std::min(a.hi, hi)}; }

// ---- elementary functions --------------------------------------------------------------------
template <class T> inline T pad_dn(T x) {
  for (int i = 0; i < ELEM_PAD_ULPS; ++i) x = std::nextafter(x, -std::numeric_limits<T>::infinity());
  return x;
}
template <class T> inline T pad_up(T x) {
  for (int i = 0; i < ELEM_PAD_ULPS; ++i) x = std::nextafter(x, std::numeric_limits<T>::infinity());
  return x;
}
// libm in double, round-to-nearest; in FP32 mode the double result is converted (rn) to float
template <class T> inline T el_sin(T x) { return T(std::sin(double(x))); }
template <class T> inline T el_cos(T x) { return T(std::cos(double(x))); }
template <class T> inline T el_atan2(T y, T x) { return T(std::atan2(double(y), double(x))); }

template <class T> struct PiC;   // outward-rounded bounds of pi and pi/2 in T
template <> struct PiC<double> {
  static constexpr double PI_LO = 0x1.921fb54442d18p+1, PI_HI = 0x1.921fb54442d19p+1;
  static constexpr double PIO2_LO = 0x1.921fb54442d18p+0, PIO2_HI = 0x1.921fb54442d19p+0;
};
template <> struct PiC<float> {
  static constexpr float PI_LO = 0x1.921fb4p+1f, PI_HI = 0x1.921fb6p+1f;
  static constexpr float PIO2_LO = 0x1.921fb4p+0f, PIO2_HI = 0x1.921fb6p+0f;
};

// enclosure of sin over e.  Outside [-4,4] (or NaN) -> [-1,1].  Inside [-4,4] the only interior
// critical points are +pi/2 (max) and -pi/2 (min).
template <class T> inline Iv<T> isin(Iv<T> e) {
  if (!(e.lo >= T(-4) && e.hi <= T(4))) return {T(-1), T(1)};
  NearestInUp rn;
  T a = el_sin(e.lo), b = el_sin(e.hi);
  Iv<T> r = {pad_dn(std::min(a, b)), pad_up(std::max(a, b))};
  if (e.lo <= PiC<T>::PIO2_HI && e.hi >= PiC<T>::PIO2_LO) r.hi = T(1);
  if (e.lo <= -PiC<T>::PIO2_LO && e.hi >= -PiC<T>::PIO2_HI) r.lo = T(-1);
  return iclamp(r, T(-1), T(1));
}
// enclosure of cos over e: interior critical points in [-4,4] are 0 (max) and +-pi (min).
template <class T> inline Iv<T> icos(Iv<T> e) {
  if (!(e.lo >= T(-4) && e.hi <= T(4))) return {T(-1), T(1)};
  NearestInUp rn;
  T a = el_cos(e.lo), b = el_cos(e.hi);
  Iv<T> r = {pad_dn(std::min(a, b)), pad_up(std::max(a, b))};
  if (e.lo <= T(0) && e.hi >= T(0)) r.hi = T(1);
  if (e.lo <= PiC<T>::PI_HI && e.hi >= PiC<T>::PI_LO) r.lo = T(-1);
  if (e.lo <= -PiC<T>::PI_LO && e.hi >= -PiC<T>::PI_HI) r.lo = T(-1);
  return iclamp(r, T(-1), T(1));
}
// enclosure of atan2(y, x) over the rectangle y x x.  The angle is monotone along every edge of a
// rectangle that avoids the cut (negative x axis) and the origin, so the extremes are at corners.
template <class T> inline Iv<T> iatan2(Iv<T> y, Iv<T> x) {
  if (x.lo <= T(0) && y.lo <= T(0) && y.hi >= T(0)) return {-PiC<T>::PI_HI, PiC<T>::PI_HI};
  NearestInUp rn;
  T c0 = el_atan2(y.lo, x.lo), c1 = el_atan2(y.lo, x.hi), c2 = el_atan2(y.hi, x.lo), c3 = el_atan2(y.hi, x.hi);
  Iv<T> r = {pad_dn(std::min(std::min(c0, c1), std::min(c2, c3))), pad_up(std::max(std::max(c0, c1), std::max(c2, c3)))};
  return iclamp(r, -PiC<T>::PI_HI, PiC<T>::PI_HI);
}

// ---- inputs ---------------------------------------------------------------------------------
struct OrcWire { double x0, y0, sin_phi_s, cos_phi_s, tan_tau; };   // (A.1a,b) L147-152
struct OrcHit { int32_t wire; int32_t pad; double drift; };         // |d_St| measured, L88
struct OrcParams { double tol, x_ref, y_ref, z_ref; int32_t precision; uint32_t flags; };

// per-hit scalars, computed once in round-to-nearest and then taken as exact (G-scalars)
template <class T> struct HitC {
  T xA, yA;        // (A.4d,e) L174-176: wire point in the plane z = z_ref
  T sphi, cphi, Tn;
  T k0, kx, ky;    // S3: cross term  k0 + ky*X + kx*Y
  T mx, my, h2;    // S3: dot term   (X-mx)^2 + (Y-my)^2 - h2
  T d, tol, zref;
  int rigorous;    // params.flags bit 4: Phi from a verified enclosure of the fixed point of (A.6) (reading f3)
  int full_turn;   // params.flags bit 3 (paper mode only): turning angles unwrapped for tracks of up to one turn (M6)
  T xr, yr;        // the reference point (M6 needs it beside the S3 scalars)
};

template <class T> HitC<T> make_hitc(const OrcWire& w, const OrcHit& h, const OrcParams& p) {
  // round-to-nearest, unfused.  In FP32 mode every scalar input is first converted to float.
  HitC<T> c;
  T x0 = T(w.x0), y0 = T(w.y0), s = T(w.sin_phi_s), co = T(w.cos_phi_s), t = T(w.tan_tau);
  T xr = T(p.x_ref), yr = T(p.y_ref), zr = T(p.z_ref);
  c.sphi = s; c.cphi = co; c.Tn = t;
  c.xA = opaque(x0 + opaque(opaque(zr * s) * t));
  c.yA = opaque(y0 - opaque(opaque(zr * co) * t));
  c.k0 = opaque(opaque(xr * c.yA) - opaque(yr * c.xA));
  c.ky = opaque(yr - c.yA);
  c.kx = opaque(c.xA - xr);
  c.mx = opaque(T(0.5) * opaque(xr + c.xA));
  c.my = opaque(T(0.5) * opaque(yr + c.yA));
  T hx = opaque(T(0.5) * opaque(c.xA - xr)), hy = opaque(T(0.5) * opaque(c.yA - yr));
  c.h2 = opaque(opaque(hx * hx) + opaque(hy * hy));
  c.d = T(h.drift); c.tol = T(p.tol); c.zref = zr;
  c.full_turn = (p.flags & 8u) ? 1 : 0;
  c.xr = xr; c.yr = yr;
  c.rigorous = (p.flags & 16u) ? 1 : 0;
  return c;
}

template <class T> struct Box { Iv<T> X, Y, R, Z, L; };

struct Resid { double flo, fhi, scale; bool decided_vote; };   // decided_vote: domain rule forced a vote

// S1-S8 for one (box, hit, drift sign).  Mode must be FE_UPWARD.  sign = +1 / -1.
template <class T> Resid residual(const Box<T>& b, const HitC<T>& c, int sign) {
  const T one = T(1), two = T(2), half = T(0.5);
  // S1 drift interval, tolerance applied on d_St before delta = d/u (G6)
  Iv<T> D = {std::max(dn_add(c.d, -c.tol), T(0)), up_add(c.d, c.tol)};
  if (sign < 0) D = ineg(D);
  // S2 transverse part (A.7a,d,e) L191-201
  Iv<T> A = isub(thin(c.xA), b.X), B = isub(thin(c.yA), b.Y);
  Iv<T> Q = iadd(isqr(A), isqr(B));
  Iv<T> cA = isub(iscale(c.sphi, A), iscale(c.cphi, B));
  Iv<T> sA = iadd(iscale(c.cphi, A), iscale(c.sphi, B));
  // S3' domain rule: the xy cell may contain the wire point -> cannot exclude (G15)
  if (!(Q.lo > T(0))) return {0.0, 0.0, double(Q.hi), true};
  // S3 turning angle phi_Ax - phi0 (1d) L49, (A.7f) L203, as one atan2(cross, dot) (G8)
  Iv<T> cr = iadd(iadd(thin(c.k0), iscale(c.ky, b.X)), iscale(c.kx, b.Y));
  Iv<T> dt = isub(iadd(isqr(isub(b.X, thin(c.mx))), isqr(isub(b.Y, thin(c.my)))), thin(c.h2));
  Iv<T> dphi = iatan2(cr, dt);
  // S3' (A.7a,g)
  Iv<T> iQ = irecip_pos(Q);
  Iv<T> RA = isqrt(Q);
  Iv<T> iR = irecip_pos(RA);
  Iv<T> c2 = imul(isub(isqr(cA), isqr(sA)), iQ);        // cos 2Phi_Ax
  Iv<T> s2 = imul(iscale(two, imul(sA, cA)), iQ);       // sin 2Phi_Ax
  // S4 series (A.8a-d) L211-218
  Iv<T> Zr = isub(b.Z, thin(c.zref));
  Iv<T> LR = imul(b.L, b.R);
  Iv<T> zA = iadd(Zr, imul(LR, dphi));                  // (A.8d)
  Iv<T> LD = imul(b.L, D);
  Iv<T> P1 = ineg(imul(iadd(imul(zA, sA), imul(LD, cA)), iQ));                         // (A.8b)
  Iv<T> t1 = imul(LR, zA);
  Iv<T> t2 = imul(imul(imul(b.L, zA), isub(b.R, iscale(two, D))), c2);
  Iv<T> t3 = imul(iadd(isqr(zA), imul(D, iadd(RA, imul(isqr(b.L), isub(iadd(b.R, RA), D))))), s2);
  Iv<T> P2 = iscale(half, imul(iadd(isub(t1, t2), t3), iQ));                           // (A.8c)
  Iv<T> T2 = isqr(thin(c.Tn));
  Iv<T> e = iadd(iscale(c.Tn, P1), imul(T2, P2));       // Phi - Phi_Ax  (A.8a)
  // S5-S7 as a function of e = Phi - Phi_Ax (they are evaluated once with the series value, or - rigorous mode -
  // several times inside the verification of the fixed point of (A.6))
  Iv<T> sinP, cosP, dl, z, Ld, ct;
  bool u_ok = true;
  auto s5_to_s7 = [&](Iv<T> ee) {
    // S5 trig of Phi = Phi_Ax + e  (A.3b), (A.7g)
    Iv<T> se = isin(ee), ce = icos(ee);
    sinP = iclamp(imul(iadd(imul(sA, ce), imul(cA, se)), iR), T(-1), one);
    cosP = iclamp(imul(isub(imul(cA, ce), imul(sA, se)), iR), T(-1), one);
    // S6 drift-line norm (A.3a) L160 and delta = d_St / u_d
    Iv<T> u2 = iadd(iadd(iadd(thin(one), iscale(opaque(two * c.Tn), imul(b.L, sinP))), imul(T2, isqr(b.L))),
                    imul(T2, isqr(cosP)));
    Iv<T> u = isqrt(u2);
    if (!(u.lo > T(0))) { u_ok = false; return; }
    dl = idiv_pos(D, u);
    // S7 z of the wire point (A.4c) L172 with s_perp = R (dphi + e);  c^tau (A.7b) L194
    z = isub(iadd(Zr, imul(LR, iadd(dphi, ee))), iscale(c.Tn, imul(dl, cosP)));
    Ld = imul(b.L, dl);
    ct = isub(imul(z, cA), imul(Ld, sA));
  };
  if (c.rigorous) {
    // Reading f3 (PAPER.md L187 eq. (A.6) "solved numerically"): e is a fixed point of
    //   g(e) = atan2( T s^tau(e), R_Ax^2 + T c^tau(e) ),  s^tau = -z s_Ax - lambda delta c_Ax   (A.6), (A.7b,c)
    // Verification by inflation: start from the series enclosure; if g(E) is inside E, g has a fixed point in
    // g(E) (Brouwer) - taken as THE solution of (A.6) on this branch - and E := g(E), then once more
    // E := g(E) meet E.  Otherwise E := hull(E, g(E)) widened by a tenth of its width (+ a small absolute
    // amount) and again, at most RIG_ROUNDS times; no verification: the hit votes (cannot exclude).
    const int RIG_ROUNDS = 6;
    const T tiny = std::is_same<T, float>::value ? T(1e-6) : T(1e-12);
    auto g_of = [&](Iv<T> ee, Iv<T>& out) -> bool {
      s5_to_s7(ee);
      if (!u_ok) return false;
      Iv<T> st = ineg(iadd(imul(z, sA), imul(Ld, cA)));
      out = iatan2(iscale(c.Tn, st), iadd(Q, iscale(c.Tn, ct)));
      return true;
    };
    Iv<T> E = e, G;
    bool verified = false;
    for (int k = 0; k < RIG_ROUNDS && !verified; ++k) {
      if (!g_of(E, G)) return {0.0, 0.0, double(Q.hi), true};
      if (G.lo >= E.lo && G.hi <= E.hi) {
        verified = true;
        E = G;
      } else {
        const T lo_h = std::min(E.lo, G.lo), hi_h = std::max(E.hi, G.hi);
        const T pad = up_add(up_mul(T(0.1), up_add(hi_h, -lo_h)), tiny);
        E = {dn_add(lo_h, -pad), up_add(hi_h, pad)};
      }
    }
    if (!verified) return {0.0, 0.0, double(Q.hi), true};
    if (!g_of(E, G)) return {0.0, 0.0, double(Q.hi), true};
    e = {std::max(E.lo, G.lo), std::min(E.hi, G.hi)};
    if (!(e.lo <= e.hi)) return {0.0, 0.0, double(Q.hi), true};
  }
  s5_to_s7(e);
  if (!u_ok) return {0.0, 0.0, double(Q.hi), true};
  // S8 (R + d_Ax)^2 = radicand of (A.5b) L183;  f = R_Ax^2 - (R + d_Ax)^2  (A.5a) L180
  Iv<T> rad = isub(isub(isub(isqr(iadd(b.R, dl)), iscale(opaque(two * c.Tn), ct)), isqr(iscale(c.Tn, z))),
                   isqr(iscale(c.Tn, Ld)));
  Iv<T> f = isub(Q, rad);
  double sc = std::max(double(Q.hi), std::max(std::fabs(double(rad.lo)), std::fabs(double(rad.hi))));
  return {double(f.lo), double(f.hi), sc, false};
}

inline bool votes_yes(const Resid& r) { return r.decided_vote || !(r.flo > 0.0 || r.fhi < 0.0); }

// one hit, one box: vote iff either drift sign cannot be excluded (G7: at most one vote per hit)
template <class T> bool hit_votes(const Box<T>& b, const HitC<T>& c) {
  return votes_yes(residual(b, c, +1)) || votes_yes(residual(b, c, -1));
}

// outward conversion of a double box edge to T
template <class T> inline T cvt_dn(double x);
template <class T> inline T cvt_up(double x);
template <> inline double cvt_dn<double>(double x) { return x; }
template <> inline double cvt_up<double>(double x) { return x; }
template <> inline float cvt_dn<float>(double x) {
  float f = float(x);   // any mode: fix up explicitly
  if (double(f) > x) f = std::nextafter(f, -std::numeric_limits<float>::infinity());
  return f;
}
template <> inline float cvt_up<float>(double x) {
  float f = float(x);
  if (double(f) < x) f = std::nextafter(f, std::numeric_limits<float>::infinity());
  return f;
}
template <class T> Box<T> make_box(const double lo[5], const double hi[5]) {
  Box<T> b;
  b.X = {cvt_dn<T>(lo[0]), cvt_up<T>(hi[0])};
  b.Y = {cvt_dn<T>(lo[1]), cvt_up<T>(hi[1])};
  b.R = {cvt_dn<T>(lo[2]), cvt_up<T>(hi[2])};
  b.Z = {cvt_dn<T>(lo[3]), cvt_up<T>(hi[3])};
  b.L = {cvt_dn<T>(lo[4]), cvt_up<T>(hi[4])};
  return b;
}

// cell edges e_k = lo + k*((hi-lo)/n), e_n = hi : round-to-nearest, unfused (S9, G14)
std::vector<double> edges(double lo, double hi, int n) {
  std::vector<double> e(n + 1);
  double w = opaque(opaque(hi - lo) / double(n));
  for (int k = 0; k < n; ++k) e[k] = opaque(lo + opaque(double(k) * w));
  e[n] = hi;
  return e;
}

enum { ORC_OK = 0, ORC_ERR_ARG = -1, ORC_ERR_GEOMETRY = -2, ORC_ERR_DOMAIN = -3 };

int check_domain(const OrcWire* wires, int n_wires, const OrcHit* hits, int n_hits, double Rlo, double Llo, double Lhi) {
  double tmax = 0;
  for (int i = 0; i < n_hits; ++i) {
    if (hits[i].wire < 0 || hits[i].wire >= n_wires) return ORC_ERR_GEOMETRY;
    if (!(hits[i].drift >= 0)) return ORC_ERR_ARG;
    tmax = std::max(tmax, std::fabs(wires[hits[i].wire].tan_tau));
  }
  if (!(Rlo > 0)) return ORC_ERR_DOMAIN;
  if (!(std::max(std::fabs(Llo), std::fabs(Lhi)) * tmax < 0.5)) return ORC_ERR_DOMAIN;
  return ORC_OK;
}

template <class T> std::vector<HitC<T>> stage_hits(const OrcWire* wires, const OrcHit* hits, int n_hits, const OrcParams& p) {
  std::vector<HitC<T>> hc(n_hits);
  for (int i = 0; i < n_hits; ++i) hc[i] = make_hitc<T>(wires[hits[i].wire], hits[i], p);
  return hc;
}

template <class T>
void vote_boxes_T(const std::vector<HitC<T>>& hc, const double* blo, const double* bhi, int64_t n_boxes, uint16_t* out) {
#pragma omp parallel
  {
    UpMode up;
#pragma omp for schedule(dynamic, 64)
    for (int64_t i = 0; i < n_boxes; ++i) {
      Box<T> b = make_box<T>(blo + 5 * i, bhi + 5 * i);
      unsigned v = 0;
      for (const auto& c : hc) v += hit_votes(b, c) ? 1u : 0u;
      out[i] = uint16_t(v);
    }
  }
}

struct Grid {
  std::vector<double> e[5];
  int n[5];
  Grid(const double lo[5], const double hi[5], const int32_t dims[5]) {
    for (int d = 0; d < 5; ++d) { n[d] = dims[d]; e[d] = edges(lo[d], hi[d], dims[d]); }
  }
  int64_t cells() const { int64_t c = 1; for (int d = 0; d < 5; ++d) c *= n[d]; return c; }
  // linear index ((((ix*ny+iy)*nR+iR)*nz+iz)*nl+il): lambda fastest (S9)
  void cell(int64_t idx, double lo[5], double hi[5]) const {
    for (int d = 4; d >= 0; --d) { int k = int(idx % n[d]); idx /= n[d]; lo[d] = e[d][k]; hi[d] = e[d][k + 1]; }
  }
};

template <class T>
void vote_cells_T(const std::vector<HitC<T>>& hc, const Grid& g, const int64_t* cell_idx, int64_t n, uint16_t* out) {
#pragma omp parallel
  {
    UpMode up;
#pragma omp for schedule(dynamic, 256)
    for (int64_t i = 0; i < n; ++i) {
      double lo[5], hi[5];
      g.cell(cell_idx ? cell_idx[i] : i, lo, hi);
      Box<T> b = make_box<T>(lo, hi);
      unsigned v = 0;
      for (const auto& c : hc) v += hit_votes(b, c) ? 1u : 0u;
      out[i] = uint16_t(v);
    }
  }
}

// key order: votes descending, index ascending (S9, G16)
void topk_plain(const uint16_t* votes, int64_t n, int k, int64_t* idx_out, uint16_t* votes_out) {
  std::vector<int64_t> idx(n);
  for (int64_t i = 0; i < n; ++i) idx[i] = i;
  auto better = [&](int64_t a, int64_t b) { return votes[a] != votes[b] ? votes[a] > votes[b] : a < b; };
  std::partial_sort(idx.begin(), idx.begin() + k, idx.end(), better);
  for (int i = 0; i < k; ++i) { idx_out[i] = idx[i]; votes_out[i] = votes[idx[i]]; }
}

struct OrcBox { double lo[5], hi[5]; uint16_t votes; uint16_t pad[3]; };

template <class T>
int refine_T(const OrcWire* wires, int n_wires, const OrcHit* hits, int n_hits, const OrcParams& p,
             const double lo[5], const double hi[5], const int32_t grid0[5], int levels, int k,
             OrcBox* boxes_out, double* params_out) {
  auto hc = stage_hits<T>(wires, hits, n_hits, p);
  Grid g(lo, hi, grid0);
  int64_t n0 = g.cells();
  if (k > n0) return ORC_ERR_ARG;
  std::vector<uint16_t> votes(n0);
  vote_cells_T<T>(hc, g, nullptr, n0, votes.data());
  std::vector<int64_t> idx(k);
  std::vector<uint16_t> kv(k);
  topk_plain(votes.data(), n0, k, idx.data(), kv.data());
  std::vector<OrcBox> cur(k);
  for (int r = 0; r < k; ++r) { g.cell(idx[r], cur[r].lo, cur[r].hi); cur[r].votes = kv[r]; std::memset(cur[r].pad, 0, sizeof cur[r].pad); }
  std::copy(cur.begin(), cur.end(), boxes_out);
  for (int lev = 1; lev < levels; ++lev) {
    // children: list index rank*32 + c; bit (4-dim) of c set -> upper half [mid, hi]; mid = 0.5*(lo+hi) rn (S9, G18)
    int64_t nc = int64_t(k) * 32;
    std::vector<double> clo(nc * 5), chi(nc * 5);
    for (int r = 0; r < k; ++r)
      for (int c = 0; c < 32; ++c)
        for (int d = 0; d < 5; ++d) {
          double mid = opaque(0.5 * opaque(cur[r].lo[d] + cur[r].hi[d]));
          bool upper = (c >> (4 - d)) & 1;
          clo[(r * 32 + c) * 5 + d] = upper ? mid : cur[r].lo[d];
          chi[(r * 32 + c) * 5 + d] = upper ? cur[r].hi[d] : mid;
        }
    std::vector<uint16_t> cv(nc);
    vote_boxes_T<T>(hc, clo.data(), chi.data(), nc, cv.data());
    topk_plain(cv.data(), nc, k, idx.data(), kv.data());
    for (int r = 0; r < k; ++r) {
      for (int d = 0; d < 5; ++d) { cur[r].lo[d] = clo[idx[r] * 5 + d]; cur[r].hi[d] = chi[idx[r] * 5 + d]; }
      cur[r].votes = kv[r];
    }
    // idx refers to the previous cur; write after all reads (clo/chi are copies, so this is safe)
    std::copy(cur.begin(), cur.end(), boxes_out + int64_t(lev) * k);
  }
  // value = centre, error = half-width of the rank-0 box of the last pass (L94, G19)
  for (int d = 0; d < 5; ++d) {
    params_out[d] = opaque(0.5 * opaque(cur[0].lo[d] + cur[0].hi[d]));
    params_out[5 + d] = opaque(0.5 * opaque(cur[0].hi[d] - cur[0].lo[d]));
  }
  // G19: "additionally report hull of last-pass boxes with votes == max" - the paper keeps ALL the cells
  // at the maximum and takes value and error from their centres and sizes (L94); of the K kept boxes those at the
  // maximum are the ones with the votes of rank 0
  for (int d = 0; d < 5; ++d) {
    double hl = cur[0].lo[d], hh = cur[0].hi[d];
    for (int r = 1; r < k; ++r)
      if (cur[r].votes == cur[0].votes) { hl = std::min(hl, cur[r].lo[d]); hh = std::max(hh, cur[r].hi[d]); }
    params_out[10 + d] = hl;
    params_out[15 + d] = hh;
  }
  return ORC_OK;
}

}  // namespace

// =============================================================================================
// Paper-mode vote: the configuration the paper ran.
//   M1  voxel = 4-D interval  xc x yc x R x z0  (L64); its mid-point m = 0.5*(lo+hi) per axis.
//   M2  "The momentum of the particle is fixed to its true value" (L64): |p| enters as the length
//       P = R sqrt(1 + lambda^2) (the radius a track of that momentum would have at lambda = 0), so
//       |lambda| = sqrt((P/R_m)^2 - 1) at the voxel's mid radius; "The sign of lambda remains unknown
//       ... This procedure is applied for each sign of the lambda value, so two 4D accumulators are
//       used" (L64, L78): accumulator 0 takes +|lambda|, accumulator 1 takes -|lambda|.  A voxel
//       with R_m > P has no lambda and gets no vote (reading M2 of DESIGN.md).
//   M3  "the variables appearing in the expression of d_Ax, given in the equation (A.5b), are not
//       considered as interval.  Their values are taken in the middle of the voxel" (L82):
//       d_Ax = sqrt(radicand of (A.5b)) - R_m from steps S2-S8 evaluated at the point
//       (xc_m, yc_m, R_m, z0_m, +-|lambda|) in plain round-to-nearest double arithmetic, same
//       association order as the interval form.  A negative radicand or a NaN: that drift sign
//       does not vote (no virtual circle exists).
//   M4  tolerance (not in the paper, L88; BASELINE's +-tol): d_Ax is evaluated at d - tol (clamped
//       at 0) and d + tol and the hull of the two values is used; tol = 0 is the paper's literal form.
//   M5  condition (4) L74-76:  0 in (x_Ax - xc)^2 + (y_Ax - yc)^2 - (R + d_Ax)^2  in interval
//       arithmetic (outward rounding), for the two drift signs; one count per hit (G7).
// The property "false => the solution is not in the voxel" is lost in this mode, as L80-82 says.
// =============================================================================================
struct PointEval { bool ok; double rad, dax; };

// S2-S8 at a point.  The caller holds FE_TONEAREST.  D is the signed drift distance.
__attribute__((noinline)) PointEval dax_point(const HitC<double>& c, double xc, double yc, double R, double z0, double lam, double D) {
  const double Tn = c.Tn;
  // S2
  const double A = c.xA - xc, B = c.yA - yc;
  const double Q = A * A + B * B;
  const double cA = A * c.sphi - B * c.cphi;
  const double sA = A * c.cphi + B * c.sphi;
  // S3
  const double cr = (c.k0 + c.ky * xc) + c.kx * yc;
  const double dx = xc - c.mx, dy = yc - c.my;
  const double dt = (dx * dx + dy * dy) - c.h2;
  double dphi = std::atan2(cr, dt);
  // reading M6 (flags bit 3): a counter-clockwise track of less than one turn (L88) emitted near the z axis (L88: at the
  // origin; L123: 5 cm from it) has turned by an angle theta in [-m, 2 pi - m) past the point of its base circle closest
  // to the axis when it reaches a given point of the circle, m = 0.3 rad.  phi_Ax - phi0 of (A.8d) is taken as
  // theta(wire point) - theta(reference point): right for every hit of such a track wherever the reference point
  // lies (it moves along the track between the passes, L98); theta(P) = atan2(cross, dot) of S3 with the reference
  // replaced by the axis and the wire point by P.  With the reference point at (0, 0) this is the S3 angle moved
  // from (-pi, pi] to [-m, 2 pi - m).
  if (c.full_turn) {
    const double two_pi = 6.283185307179586, m = 0.3;
    auto theta = [&](double px, double py) {
      const double hx = 0.5 * px, hy = 0.5 * py;
      const double cr0 = (0.0 - py) * xc + px * yc;
      const double ex = xc - hx, ey = yc - hy;
      const double dt0 = (ex * ex + ey * ey) - (hx * hx + hy * hy);
      double th = std::atan2(cr0, dt0);
      if (th < -m) th = th + two_pi;
      return th;
    };
    dphi = theta(c.xA, c.yA) - theta(c.xr, c.yr);
  }
  // S3'
  const double iQ = 1.0 / Q, RA = std::sqrt(Q), iR = 1.0 / RA;
  const double c2 = (cA * cA - sA * sA) * iQ;
  const double s2 = (2.0 * (sA * cA)) * iQ;
  // S4
  const double Zr = z0 - c.zref;
  const double LR = lam * R;
  const double zA = Zr + LR * dphi;
  const double LD = lam * D;
  const double P1 = -((zA * sA + LD * cA) * iQ);
  const double t1 = LR * zA;
  const double t2 = ((lam * zA) * (R - 2.0 * D)) * c2;
  const double t3 = (zA * zA + D * (RA + (lam * lam) * ((R + RA) - D))) * s2;
  const double P2 = 0.5 * (((t1 - t2) + t3) * iQ);
  const double T2 = Tn * Tn;
  const double e = Tn * P1 + T2 * P2;
  // S5
  const double se = std::sin(e), ce = std::cos(e);
  double sinP = (sA * ce + cA * se) * iR, cosP = (cA * ce - sA * se) * iR;
  sinP = std::min(1.0, std::max(-1.0, sinP));
  cosP = std::min(1.0, std::max(-1.0, cosP));
  // S6
  const double u2 = ((1.0 + (2.0 * Tn) * (lam * sinP)) + T2 * (lam * lam)) + T2 * (cosP * cosP);
  const double u = std::sqrt(u2);
  const double dl = D / u;
  // S7
  const double z = (Zr + LR * (dphi + e)) - Tn * (dl * cosP);
  const double Ld = lam * dl;
  const double ct = z * cA - Ld * sA;
  // S8
  const double Rd = R + dl, Tz = Tn * z, TLd = Tn * Ld;
  const double rad = ((Rd * Rd - (2.0 * Tn) * ct) - Tz * Tz) - TLd * TLd;
  if (!(rad >= 0.0)) return {false, rad, 0.0};
  return {true, rad, std::sqrt(rad) - R};
}

struct PaperResid { double flo, fhi, scale; bool has; };   // has = false: no d_Ax for this sign -> no vote

// M3-M4: hull of d_Ax at d - tol and d + tol, at the voxel's mid-point.  Switches to FE_TONEAREST for
// its own duration; noinline and fenced so that no operation drifts across the mode switches.
__attribute__((noinline)) bool paper_dax_hull(const double lo[4], const double hi[4], const HitC<double>& c, double lam,
                                              int dsign, double* dax0, double* dax1) {
  NearestInUp rn;
  asm volatile("" ::: "memory");
  double m[4];
  for (int d = 0; d < 4; ++d) m[d] = opaque(0.5 * opaque(lo[d] + hi[d]));
  const double dlo = std::max(opaque(c.d - c.tol), 0.0), dhi = opaque(c.d + c.tol);
  const PointEval a = dax_point(c, m[0], m[1], m[2], m[3], lam, dsign > 0 ? dlo : -dlo);
  const PointEval b = dax_point(c, m[0], m[1], m[2], m[3], lam, dsign > 0 ? dhi : -dhi);
  bool ok = a.ok && b.ok;
  *dax0 = opaque(std::min(a.dax, b.dax));
  *dax1 = opaque(std::max(a.dax, b.dax));
  asm volatile("" ::: "memory");
  return ok;
}

// M3-M5 for one (voxel, hit, lambda sign, drift sign).  Mode must be FE_UPWARD.
PaperResid paper_residual(const double lo[4], const double hi[4], const HitC<double>& c, double lam, int dsign) {
  double dax0, dax1;
  if (!paper_dax_hull(lo, hi, c, lam, dsign, &dax0, &dax1)) return {0.0, 0.0, 0.0, false};
  const Iv<double> X = {lo[0], hi[0]}, Y = {lo[1], hi[1]}, R = {lo[2], hi[2]}, Dax = {dax0, dax1};
  const Iv<double> Q = iadd(isqr(isub(thin(c.xA), X)), isqr(isub(thin(c.yA), Y)));
  const Iv<double> S = isqr(iadd(R, Dax));
  const Iv<double> f = isub(Q, S);
  return {f.lo, f.hi, std::max(Q.hi, S.hi), true};
}

// |lambda| of the voxel from the fixed momentum (M2); false if R_m > P
__attribute__((noinline)) bool paper_lambda(double Rlo, double Rhi, double P, double* lam) {
  NearestInUp rn;
  asm volatile("" ::: "memory");
  const double Rm = opaque(0.5 * opaque(Rlo + Rhi));
  const double q = opaque(P / Rm);
  const double l2 = opaque(opaque(q * q) - 1.0);
  const bool ok = l2 >= 0.0;
  *lam = ok ? opaque(std::sqrt(l2)) : 0.0;
  asm volatile("" ::: "memory");
  return ok;
}

struct Grid4 {
  std::vector<double> e[4];
  int n[4];
  Grid4(const double lo[4], const double hi[4], const int32_t dims[4]) {
    for (int d = 0; d < 4; ++d) { n[d] = dims[d]; e[d] = edges(lo[d], hi[d], dims[d]); }
  }
  int64_t cells() const { int64_t c = 1; for (int d = 0; d < 4; ++d) c *= n[d]; return c; }
  // linear index (((ix*ny+iy)*nR+iR)*nz+iz): z0 fastest
  void cell(int64_t idx, double lo[4], double hi[4]) const {
    for (int d = 3; d >= 0; --d) { int k = int(idx % n[d]); idx /= n[d]; lo[d] = e[d][k]; hi[d] = e[d][k + 1]; }
  }
};

// ---- paper's iteration scheme, pieces -----------
// F2a  disk pre-filter, conditions (3a),(3b) L66-70: a voxel is considered only if
//        0 in xc^2 + yc^2 - (R + R_Disk)^2,   R_Disk = [-r_disk, +r_disk]
//      (the particle is emitted within r_disk of the origin).  Interval arithmetic, outward rounding;
//      every variable occurs once, so the enclosure is the exact range.  Mode must be FE_UPWARD.
bool disk_passes(const double lo[4], const double hi[4], double r_disk) {
  const Iv<double> X = {lo[0], hi[0]}, Y = {lo[1], hi[1]}, R = {lo[2], hi[2]}, D = {-r_disk, r_disk};
  const Iv<double> f = isub(iadd(isqr(X), isqr(Y)), isqr(iadd(R, D)));
  return !(f.lo > 0.0 || f.hi < 0.0);
}

// F2b  selection, L94 ("voxels corresponding to selected cells where the maximum of votes in the
//      accumulator are found.  The central values and the size of the selected voxels are used to
//      calculate the parameter values with their errors") and L121 (the sign of lambda from the two
//      accumulators).  Reading (F2b): vmax = largest count in either accumulator; the sign of
//      lambda = the accumulator that holds it (both: lambda >= 0 wins); selected = the voxels of that
//      accumulator with count == vmax; value_d = centre of the mean cell index, error_d = half the extent
//      of the selected voxels along axis d.  Integer sums, so the result does not depend on any order:
//        mean index  m_d = (2 sum(k_d) + n_sel) / (2 n_sel)   (one correctly rounded division)
//        value_d = lo_d + m_d * w_d,  w_d = (hi_d - lo_d)/n_d   (rn, unfused)
//        error_d = 0.5 * ((kmax_d - kmin_d + 1) * w_d)
struct OrcPaperFit {
  double value[4], error[4];
  double lambda;          // signed, from the fixed momentum at value[2]; 0 if value[2] > P
  int32_t lambda_sign;    // +1 / -1
  int32_t vmax;
  int64_t n_sel;
  double x_ref, y_ref;    // the reference point the pass was voted with (reading F2d': it moves between passes, L98)
  double z0_centre;       // the previous pass's z0 re-expressed for this pass's reference point (centre of a z0 window)
};

// =============================================================================================
// C ABI (ctypes)
// =============================================================================================
extern "C" {

int orc_pad_ulps() { return ELEM_PAD_ULPS; }
int orc_max_threads() {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}
void orc_set_threads(int n) {
#ifdef _OPENMP
  if (n > 0) omp_set_num_threads(n);
#endif
}

// interval primitive on doubles or floats (prec 64/32), for the primitive pins.
// op: 0 add 1 sub 2 mul 3 sqr(a) 4 div_pos 5 sqrt(a) 6 sin(a) 7 cos(a) 8 atan2(a=y,b=x) 9 recip_pos(a) 10 scale(c=b.lo, a)
int orc_prim(int op, int prec, double alo, double ahi, double blo, double bhi, double* out) {
  UpMode up;
  auto run = [&](auto tag) -> int {
    using T = decltype(tag);
    Iv<T> a = {T(alo), T(ahi)}, b = {T(blo), T(bhi)}, r{};
    switch (op) {
      case 0: r = iadd(a, b); break;
      case 1: r = isub(a, b); break;
      case 2: r = imul(a, b); break;
      case 3: r = isqr(a); break;
      case 4: r = idiv_pos(a, b); break;
      case 5: r = isqrt(a); break;
      case 6: r = isin(a); break;
      case 7: r = icos(a); break;
      case 8: r = iatan2(a, b); break;
      case 9: r = irecip_pos(a); break;
      case 10: r = iscale(T(blo), a); break;
      default: return ORC_ERR_ARG;
    }
    out[0] = double(r.lo); out[1] = double(r.hi);
    return int(ORC_OK);
  };
  return prec == 32 ? run(float()) : run(double());
}

// f enclosure for every (box, hit, sign): out[((i*n_hits + h)*2 + s)*4 + {0,1,2,3}] = f.lo, f.hi, scale, decided
// sign index 0 = +, 1 = -.
int orc_residual(const OrcWire* wires, int n_wires, const OrcHit* hits, int n_hits, const OrcParams* p,
                 const double* blo, const double* bhi, int64_t n_boxes, double* out) {
  if (!wires || !hits || !p || !blo || !bhi || !out || n_hits < 0 || n_boxes < 0) return ORC_ERR_ARG;
  for (int i = 0; i < n_hits; ++i) if (hits[i].wire < 0 || hits[i].wire >= n_wires) return ORC_ERR_GEOMETRY;
  auto run = [&](auto tag) {
    using T = decltype(tag);
    auto hc = stage_hits<T>(wires, hits, n_hits, *p);
    UpMode up;
    for (int64_t i = 0; i < n_boxes; ++i) {
      Box<T> b = make_box<T>(blo + 5 * i, bhi + 5 * i);
      for (int h = 0; h < n_hits; ++h)
        for (int s = 0; s < 2; ++s) {
          Resid r = residual(b, hc[h], s == 0 ? +1 : -1);
          double* o = out + ((i * n_hits + h) * 2 + s) * 4;
          o[0] = r.flo; o[1] = r.fhi; o[2] = r.scale; o[3] = r.decided_vote ? 1.0 : 0.0;
        }
    }
  };
  if (p->precision == 32) run(float()); else run(double());
  return ORC_OK;
}

int orc_vote_boxes(const OrcWire* wires, int n_wires, const OrcHit* hits, int n_hits, const OrcParams* p,
                   const double* blo, const double* bhi, int64_t n_boxes, uint16_t* votes_out) {
  if (!wires || !hits || !p || !blo || !bhi || !votes_out || n_hits < 0 || n_boxes < 0) return ORC_ERR_ARG;
  for (int i = 0; i < n_hits; ++i) if (hits[i].wire < 0 || hits[i].wire >= n_wires) return ORC_ERR_GEOMETRY;
  if (p->precision == 32) vote_boxes_T<float>(stage_hits<float>(wires, hits, n_hits, *p), blo, bhi, n_boxes, votes_out);
  else vote_boxes_T<double>(stage_hits<double>(wires, hits, n_hits, *p), blo, bhi, n_boxes, votes_out);
  return ORC_OK;
}

// dense grid; cell_idx == NULL: all prod(dims) cells in linear order, else the listed cells only
int orc_vote(const OrcWire* wires, int n_wires, const OrcHit* hits, int n_hits, const OrcParams* p,
             const double* lo, const double* hi, const int32_t* dims, const int64_t* cell_idx, int64_t n_idx,
             uint16_t* votes_out) {
  if (!wires || !hits || !p || !lo || !hi || !dims || !votes_out || n_hits < 0) return ORC_ERR_ARG;
  for (int d = 0; d < 5; ++d) if (dims[d] <= 0 || !(hi[d] > lo[d])) return ORC_ERR_ARG;
  int rc = check_domain(wires, n_wires, hits, n_hits, lo[2], lo[4], hi[4]);
  if (rc) return rc;
  Grid g(lo, hi, dims);
  int64_t n = cell_idx ? n_idx : g.cells();
  if (cell_idx) for (int64_t i = 0; i < n; ++i) if (cell_idx[i] < 0 || cell_idx[i] >= g.cells()) return ORC_ERR_ARG;
  if (p->precision == 32) vote_cells_T<float>(stage_hits<float>(wires, hits, n_hits, *p), g, cell_idx, n, votes_out);
  else vote_cells_T<double>(stage_hits<double>(wires, hits, n_hits, *p), g, cell_idx, n, votes_out);
  return ORC_OK;
}

// boxes of listed dense cells (host plumbing for tests)
int orc_cell_boxes(const double* lo, const double* hi, const int32_t* dims, const int64_t* cell_idx, int64_t n,
                   double* blo, double* bhi) {
  Grid g(lo, hi, dims);
  for (int64_t i = 0; i < n; ++i) g.cell(cell_idx[i], blo + 5 * i, bhi + 5 * i);
  return ORC_OK;
}

int orc_topk(const uint16_t* votes, int64_t n, int k, int64_t* idx_out, uint16_t* votes_out) {
  if (!votes || !idx_out || !votes_out || k <= 0 || k > n) return ORC_ERR_ARG;
  topk_plain(votes, n, k, idx_out, votes_out);
  return ORC_OK;
}

int orc_refine(const OrcWire* wires, int n_wires, const OrcHit* hits, int n_hits, const OrcParams* p,
               const double* lo, const double* hi, const int32_t* grid0, int levels, int k,
               OrcBox* boxes_out, double* params_out) {
  if (!wires || !hits || !p || !lo || !hi || !grid0 || !boxes_out || !params_out || levels < 1 || k < 1) return ORC_ERR_ARG;
  for (int d = 0; d < 5; ++d) if (grid0[d] <= 0 || !(hi[d] > lo[d])) return ORC_ERR_ARG;
  int rc = check_domain(wires, n_wires, hits, n_hits, lo[2], lo[4], hi[4]);
  if (rc) return rc;
  if (p->precision == 32) return refine_T<float>(wires, n_wires, hits, n_hits, *p, lo, hi, grid0, levels, k, boxes_out, params_out);
  return refine_T<double>(wires, n_wires, hits, n_hits, *p, lo, hi, grid0, levels, k, boxes_out, params_out);
}

// events in CSR: hits of event e are hits[hit_offsets[e] .. hit_offsets[e+1])
int orc_refine_batch(const OrcWire* wires, int n_wires, const OrcHit* hits, const int32_t* hit_offsets, int n_events,
                     const OrcParams* p, const double* lo, const double* hi, const int32_t* grid0, int levels, int k,
                     OrcBox* boxes_out, double* params_out) {
  if (!hit_offsets || n_events < 0) return ORC_ERR_ARG;
  for (int e = 0; e < n_events; ++e) {
    int rc = orc_refine(wires, n_wires, hits + hit_offsets[e], hit_offsets[e + 1] - hit_offsets[e], p, lo, hi, grid0,
                        levels, k, boxes_out + int64_t(e) * levels * k, params_out + int64_t(e) * 20);
    if (rc) return rc;
  }
  return ORC_OK;
}

// ---- paper mode (f1) ------------------------------------------------------------------------------
// point evaluation for the pins: out[0] = radicand of (A.5b), out[1] = d_Ax, returns 1 if no d_Ax exists
int orc_dax_point(const OrcWire* wire, const OrcParams* p, const double pt[5], double D_signed, double* out) {
  if (!wire || !p || !pt || !out) return ORC_ERR_ARG;
  OrcHit h = {0, 0, std::fabs(D_signed)};
  HitC<double> c = make_hitc<double>(*wire, h, *p);
  UpMode up;
  PointEval r;
  {
    NearestInUp rn;
    asm volatile("" ::: "memory");
    r = dax_point(c, pt[0], pt[1], pt[2], pt[3], pt[4], D_signed);
    asm volatile("" ::: "memory");
  }
  out[0] = r.rad; out[1] = r.dax;
  return r.ok ? 0 : 1;
}

// f enclosure of condition (4) for every (voxel, hit, lambda sign, drift sign):
// out[(((i*n_hits + h)*2 + ls)*2 + ds)*4 + {0,1,2,3}] = f.lo, f.hi, scale, has (0: no d_Ax or no lambda -> no vote)
int orc_residual_paper(const OrcWire* wires, int n_wires, const OrcHit* hits, int n_hits, const OrcParams* p, double P,
                       const double* blo, const double* bhi, int64_t n_boxes, double* out) {
  if (!wires || !hits || !p || !blo || !bhi || !out || n_hits < 0 || !(P > 0)) return ORC_ERR_ARG;
  for (int i = 0; i < n_hits; ++i) if (hits[i].wire < 0 || hits[i].wire >= n_wires) return ORC_ERR_GEOMETRY;
  std::vector<HitC<double>> hc = stage_hits<double>(wires, hits, n_hits, *p);
  UpMode up;
  for (int64_t i = 0; i < n_boxes; ++i) {
    const double* lo = blo + 4 * i; const double* hi = bhi + 4 * i;
    double lam = 0;
    const bool has_l = paper_lambda(lo[2], hi[2], P, &lam);
    for (int h = 0; h < n_hits; ++h)
      for (int ls = 0; ls < 2; ++ls)
        for (int ds = 0; ds < 2; ++ds) {
          PaperResid r = {0, 0, 0, false};
          if (has_l) r = paper_residual(lo, hi, hc[h], ls == 0 ? lam : -lam, ds == 0 ? +1 : -1);
          double* o = out + ((((i * n_hits + h) * 2 + ls) * 2 + ds) * 4);
          o[0] = r.flo; o[1] = r.fhi; o[2] = r.scale; o[3] = r.has ? 1.0 : 0.0;
        }
  }
  return ORC_OK;
}

// dense 4-D grid, two accumulators: votes_out[ls*n + i], ls = 0 for lambda >= 0, 1 for lambda < 0;
// cell_idx == NULL: all prod(dims) voxels in linear order (z0 fastest), else the listed voxels
// hit_mask (may be NULL): hits with mask 0 are not used (L96: "Only the selected hits are used for the next
// iteration"); r_disk >= 0: voxels failing the disk pre-filter (3a,b) get no vote; r_disk < 0: no filter
int orc_vote_paper(const OrcWire* wires, int n_wires, const OrcHit* hits, int n_hits, const uint8_t* hit_mask,
                   const OrcParams* p, double P, double r_disk,
                   const double* lo, const double* hi, const int32_t* dims, const int64_t* cell_idx, int64_t n_idx,
                   uint16_t* votes_out) {
  if (!wires || !hits || !p || !lo || !hi || !dims || !votes_out || n_hits < 0 || !(P > 0)) return ORC_ERR_ARG;
  for (int d = 0; d < 4; ++d) if (dims[d] <= 0 || !(hi[d] > lo[d])) return ORC_ERR_ARG;
  if (!(lo[2] > 0)) return ORC_ERR_DOMAIN;
  for (int i = 0; i < n_hits; ++i) {
    if (hits[i].wire < 0 || hits[i].wire >= n_wires) return ORC_ERR_GEOMETRY;
    if (!(hits[i].drift >= 0)) return ORC_ERR_ARG;
  }
  Grid4 g(lo, hi, dims);
  const int64_t n = cell_idx ? n_idx : g.cells();
  if (cell_idx) for (int64_t i = 0; i < n; ++i) if (cell_idx[i] < 0 || cell_idx[i] >= g.cells()) return ORC_ERR_ARG;
  std::vector<HitC<double>> hc = stage_hits<double>(wires, hits, n_hits, *p);
#pragma omp parallel
  {
    UpMode up;
#pragma omp for schedule(dynamic, 256)
    for (int64_t i = 0; i < n; ++i) {
      double clo[4], chi[4];
      g.cell(cell_idx ? cell_idx[i] : i, clo, chi);
      double lam = 0;
      const bool has_l = paper_lambda(clo[2], chi[2], P, &lam) && (r_disk < 0.0 || disk_passes(clo, chi, r_disk));
      for (int ls = 0; ls < 2; ++ls) {
        unsigned v = 0;
        if (has_l)
          for (int h = 0; h < n_hits; ++h) {
            if (hit_mask && !hit_mask[h]) continue;
            const auto& c = hc[h];
            bool yes = false;
            for (int ds = 0; ds < 2 && !yes; ++ds) {
              const PaperResid r = paper_residual(clo, chi, c, ls == 0 ? lam : -lam, ds == 0 ? +1 : -1);
              yes = r.has && !(r.flo > 0.0 || r.fhi < 0.0);
            }
            v += yes ? 1u : 0u;
          }
        votes_out[int64_t(ls) * n + i] = uint16_t(v);
      }
    }
  }
  return ORC_OK;
}

int orc_cell_boxes4(const double* lo, const double* hi, const int32_t* dims, const int64_t* cell_idx, int64_t n,
                    double* blo, double* bhi) {
  Grid4 g(lo, hi, dims);
  for (int64_t i = 0; i < n; ++i) g.cell(cell_idx[i], blo + 4 * i, bhi + 4 * i);
  return ORC_OK;
}

int orc_disk_filter(const double* lo, const double* hi, const int32_t* dims, double r_disk, const int64_t* cell_idx,
                    int64_t n_idx, uint8_t* out) {
  if (!lo || !hi || !dims || !out || !(r_disk >= 0)) return ORC_ERR_ARG;
  Grid4 g(lo, hi, dims);
  const int64_t n = cell_idx ? n_idx : g.cells();
  UpMode up;
  for (int64_t i = 0; i < n; ++i) {
    double clo[4], chi[4];
    g.cell(cell_idx ? cell_idx[i] : i, clo, chi);
    out[i] = disk_passes(clo, chi, r_disk) ? 1 : 0;
  }
  return ORC_OK;
}

// which: 0 = the accumulator holding the larger maximum (ties: lambda >= 0); +1 / -1 = that accumulator
int orc_select_max_paper(const uint16_t* votes, const double* lo, const double* hi, const int32_t* dims, double P,
                         int which, OrcPaperFit* out) {
  if (!votes || !lo || !hi || !dims || !out || !(P > 0)) return ORC_ERR_ARG;
  int64_t n = 1;
  for (int d = 0; d < 4; ++d) { if (dims[d] <= 0 || !(hi[d] > lo[d])) return ORC_ERR_ARG; n *= dims[d]; }
  int vmax[2] = {0, 0};
  for (int s = 0; s < 2; ++s) for (int64_t i = 0; i < n; ++i) vmax[s] = std::max(vmax[s], int(votes[s * n + i]));
  const int s = which > 0 ? 0 : (which < 0 ? 1 : (vmax[1] > vmax[0] ? 1 : 0));
  int64_t sum[4] = {0, 0, 0, 0}, kmin[4], kmax[4], cnt = 0;
  for (int d = 0; d < 4; ++d) { kmin[d] = dims[d]; kmax[d] = -1; }
  for (int64_t i = 0; i < n; ++i) {
    if (votes[s * n + i] != vmax[s]) continue;
    int64_t idx = i;
    for (int d = 3; d >= 0; --d) {
      const int64_t k = idx % dims[d]; idx /= dims[d];
      sum[d] += k; kmin[d] = std::min(kmin[d], k); kmax[d] = std::max(kmax[d], k);
    }
    ++cnt;
  }
  for (int d = 0; d < 4; ++d) {
    const double w = opaque(opaque(hi[d] - lo[d]) / double(dims[d]));
    const double m = opaque(double(2 * sum[d] + cnt) / double(2 * cnt));
    out->value[d] = opaque(lo[d] + opaque(m * w));
    out->error[d] = opaque(0.5 * opaque(double(kmax[d] - kmin[d] + 1) * w));
  }
  const double q = opaque(P / out->value[2]);
  const double l2 = opaque(opaque(q * q) - 1.0);
  out->lambda = l2 >= 0.0 ? (s == 0 ? std::sqrt(l2) : -std::sqrt(l2)) : 0.0;
  out->lambda_sign = s == 0 ? +1 : -1;
  out->vmax = vmax[s];
  out->n_sel = cnt;
  out->x_ref = out->y_ref = out->z0_centre = 0.0;   // set by the caller that knows the reference point (orc_track_paper)
  return ORC_OK;
}

// F2c  hit finding, L96: one multidimensional interval [lo, hi] (the caller builds it: value -/+ 5 error);
//      "One hit is selected when the condition (4) is true for this multidimensional interval": paper-mode
//      condition (4) with d_Ax at the interval's mid-point, the given sign of lambda, either drift sign.
int orc_find_hits_paper(const OrcWire* wires, int n_wires, const OrcHit* hits, int n_hits, const OrcParams* p, double P,
                        int lambda_sign, const double* lo, const double* hi, uint8_t* flags_out) {
  if (!wires || !hits || !p || !lo || !hi || !flags_out || n_hits < 0 || !(P > 0)) return ORC_ERR_ARG;
  for (int d = 0; d < 4; ++d) if (!(hi[d] > lo[d])) return ORC_ERR_ARG;
  for (int i = 0; i < n_hits; ++i) if (hits[i].wire < 0 || hits[i].wire >= n_wires) return ORC_ERR_GEOMETRY;
  std::vector<HitC<double>> hc = stage_hits<double>(wires, hits, n_hits, *p);
  UpMode up;
  double lam = 0;
  const bool has_l = paper_lambda(lo[2], hi[2], P, &lam);
  for (int h = 0; h < n_hits; ++h) {
    bool yes = false;
    for (int ds = 0; ds < 2 && has_l && !yes; ++ds) {
      const PaperResid r = paper_residual(lo, hi, hc[h], lambda_sign >= 0 ? lam : -lam, ds == 0 ? +1 : -1);
      yes = r.has && !(r.flo > 0.0 || r.fhi < 0.0);
    }
    flags_out[h] = yes ? 1 : 0;
  }
  return ORC_OK;
}

// F2d' the reference-point update, L98: "In the second step, the reference point is taken as the position of
//      measurement point closest to the recovered circle. ... In the third step, a new reference point is defined as
//      in the previous step."  Reading: measurement points = the hits the previous pass's hit finding
//      selected (mask != 0; "only the selected hits are used for the next iteration", L96); position of a measurement
//      point = the wire's point in the transverse plane z = z_ref, (x_Ax, y_Ax) of (A.4d,e) - the transverse position the
//      vote itself gives the wire; distance to the recovered circle = | sqrt((x_Ax - xc)^2 + (y_Ax - yc)^2) - R | with
//      (xc, yc, R) the previous pass's values; round-to-nearest double, unfused; ties: the lowest hit index; no
//      selected hit: the reference point stays.  Returns the chosen hit index (-1: none), out_xy = the new point.
//      z0 keeps its meaning "z where the helix is closest to the reference point" (eq. (1d)), so after a move
//      it refers to the new point, and "the value determined by the previous step" on which a window is centred (L98)
//      is re-expressed for it: z0' = z0 + (lambda R) (theta(new point) - theta(old point)) with the previous pass's
//      xc, yc, R, lambda (orc_transport_z0 below; the arc between two hits times lambda can exceed the +-40 cm window).
int orc_move_ref_paper(const OrcWire* wires, int n_wires, const OrcHit* hits, int n_hits, const uint8_t* mask,
                       const OrcParams* p, const OrcPaperFit* prev, double* out_xy) {
  if (!wires || !hits || !p || !prev || !out_xy || n_hits < 0) return ORC_ERR_ARG;
  out_xy[0] = p->x_ref; out_xy[1] = p->y_ref;
  int best = -1;
  double best_d = 0.0;
  for (int h = 0; h < n_hits; ++h) {
    if (mask && !mask[h]) continue;
    if (hits[h].wire < 0 || hits[h].wire >= n_wires) return ORC_ERR_GEOMETRY;
    const OrcWire& w = wires[hits[h].wire];
    const double xA = opaque(w.x0 + opaque(opaque(p->z_ref * w.sin_phi_s) * w.tan_tau));      // (A.4d) L174
    const double yA = opaque(w.y0 - opaque(opaque(p->z_ref * w.cos_phi_s) * w.tan_tau));      // (A.4e) L176
    const double dx = opaque(xA - prev->value[0]), dy = opaque(yA - prev->value[1]);
    const double rho = std::sqrt(opaque(opaque(dx * dx) + opaque(dy * dy)));
    const double d = std::fabs(opaque(rho - prev->value[2]));
    if (best < 0 || d < best_d) { best = h; best_d = d; out_xy[0] = xA; out_xy[1] = yA; }
  }
  return best;
}

// z0 of `prev` re-expressed for the reference point (x_new, y_new): turning angles theta as in dax_point - with flags
// bit 3 counted from the point of the circle closest to the axis in [-0.3, 2 pi - 0.3) (reading M6), else the principal
// value of eq. (1d)'s phi0, their difference wrapped into (-pi, pi].  Round-to-nearest double, unfused.
double orc_transport_z0(const OrcParams* p, const OrcPaperFit* prev, double x_new, double y_new) {
  const double xc = prev->value[0], yc = prev->value[1], two_pi = 6.283185307179586;
  double dth;
  if (p->flags & 8u) {
    auto theta = [&](double px, double py) {
      const double hx = opaque(0.5 * px), hy = opaque(0.5 * py);
      const double cr0 = opaque(opaque(opaque(0.0 - py) * xc) + opaque(px * yc));
      const double ex = opaque(xc - hx), ey = opaque(yc - hy);
      const double dt0 = opaque(opaque(opaque(ex * ex) + opaque(ey * ey)) - opaque(opaque(hx * hx) + opaque(hy * hy)));
      double th = std::atan2(cr0, dt0);
      if (th < -0.3) th = opaque(th + two_pi);
      return th;
    };
    dth = opaque(theta(x_new, y_new) - theta(prev->x_ref, prev->y_ref));
  } else {
    dth = opaque(std::atan2(opaque(x_new - xc), opaque(yc - y_new)) - std::atan2(opaque(prev->x_ref - xc), opaque(yc - prev->y_ref)));
    if (dth > 3.141592653589793) dth = opaque(dth - two_pi);
    if (dth <= -3.141592653589793) dth = opaque(dth + two_pi);
  }
  return opaque(prev->value[3] + opaque(opaque(prev->lambda * prev->value[2]) * dth));
}

// F2e  the iteration scheme, L92-106: n_passes vote passes; pass i votes its grid with the hits found by the
//      previous pass (L96), selects the maximum-vote voxels (L94) and finds the hits of the next pass on
//      value -/+ factor*error.  A pass is either a fixed grid [lo, hi] x dims (Table 1, iterations 1-2) or
//      a window of half-widths `lo` (sic) around the previous pass's value (iteration 3).
//      "This procedure is applied for each sign of the lambda value" (L78): reading F2e - one chain per
//      sign of lambda (accumulator s of every pass, hits found with that sign); the sign is decided by
//      comparing the maxima of the last pass (L121; ties: lambda >= 0).  A pass with move_ref != 0 (not the
//      first) is voted with the reference point of F2d' taken from the previous pass of its chain; every fit
//      records the reference point of its pass.
struct OrcPaperPass { double lo[4], hi[4]; int32_t dims[4]; int32_t windowed; int32_t move_ref; };

int orc_track_paper(const OrcWire* wires, int n_wires, const OrcHit* hits, int n_hits, const OrcParams* p, double P,
                    double r_disk, double factor, const OrcPaperPass* passes, int n_passes, OrcPaperFit* fits_out,
                    int32_t* sign_out) {
  if (!passes || n_passes < 1 || !fits_out || !sign_out || !(factor > 0)) return ORC_ERR_ARG;
  if (passes[0].windowed || passes[0].move_ref) return ORC_ERR_ARG;
  for (int s = 0; s < 2; ++s) {
    std::vector<uint8_t> mask(n_hits, 1);
    OrcPaperFit prev{};
    OrcParams pp = *p;                       // the chain's own reference point
    for (int i = 0; i < n_passes; ++i) {
      if (passes[i].move_ref) {
        double xy[2];
        const int rc_m = orc_move_ref_paper(wires, n_wires, hits, n_hits, mask.data(), &pp, &prev, xy);
        if (rc_m < -1) return rc_m;
        pp.x_ref = xy[0]; pp.y_ref = xy[1];
      }
      // the previous z0 seen from this pass's reference point (unchanged point: unchanged value)
      const double z0c = i == 0 ? 0.0 : ((pp.x_ref == prev.x_ref && pp.y_ref == prev.y_ref) ? prev.value[3]
                                                                                             : orc_transport_z0(&pp, &prev, pp.x_ref, pp.y_ref));
      double lo[4], hi[4];
      for (int d = 0; d < 4; ++d) {
        if (passes[i].windowed) {
          const double centre = d == 3 ? z0c : prev.value[d];
          lo[d] = opaque(centre - passes[i].lo[d]);
          hi[d] = opaque(centre + passes[i].lo[d]);
        } else {
          lo[d] = passes[i].lo[d];
          hi[d] = passes[i].hi[d];
        }
      }
      int64_t n = 1;
      for (int d = 0; d < 4; ++d) n *= passes[i].dims[d];
      std::vector<uint16_t> votes(2 * n);
      int rc = orc_vote_paper(wires, n_wires, hits, n_hits, mask.data(), &pp, P, r_disk, lo, hi, passes[i].dims, nullptr, 0,
                              votes.data());
      if (rc) return rc;
      OrcPaperFit fit;
      rc = orc_select_max_paper(votes.data(), lo, hi, passes[i].dims, P, s == 0 ? +1 : -1, &fit);
      if (rc) return rc;
      fit.x_ref = pp.x_ref; fit.y_ref = pp.y_ref; fit.z0_centre = z0c;
      fits_out[i * 2 + s] = fit;
      double blo[4], bhi[4];
      for (int d = 0; d < 4; ++d) {
        const double e = opaque(factor * fit.error[d]);
        blo[d] = opaque(fit.value[d] - e);
        bhi[d] = opaque(fit.value[d] + e);
      }
      rc = orc_find_hits_paper(wires, n_wires, hits, n_hits, &pp, P, s == 0 ? +1 : -1, blo, bhi, mask.data());
      if (rc) return rc;
      prev = fit;
    }
  }
  const OrcPaperFit* last = fits_out + (n_passes - 1) * 2;
  *sign_out = last[1].vmax > last[0].vmax ? -1 : +1;
  return ORC_OK;
}

}  // extern "C"
