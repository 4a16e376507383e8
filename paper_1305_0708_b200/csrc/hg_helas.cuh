// hg_helas.cuh -- device wavefunction / vertex function library (layer L2' of SURVEY.md section 1).
//
// Same ROLES and names as the paper's HEGET functions (section 4; Appendix C), whose
// listings did not survive extraction (SURVEY.md "State of the reference text"), so every routine is
// re-derived here from the definitions (Eq. 29-34) and the Lagrangians (Eq. 35, 39, 40, 47, 50-53).
//
// Conventions (derived in DESIGN.md "Sign rule"):
//   * chiral (Weyl) representation, gamma5 = diag(-1,-1,+1,+1) (reading SURVEY.md 8c-A1):
//        gamma^mu = [[0, sigma^mu], [sigmabar^mu, 0]],  Vslash = [[0, V0 - V.sigma], [V0 + V.sigma, 0]];
//     a column spinor psi has slots A = (c0,c1) = left-handed part, B = (c2,c3) = right-handed part;
//     a row spinor psibar = psi^dagger gamma^0 has slots A = conj(right part), B = conj(left part);
//   * i M = prod(i V_vertex) prod(i P_propagator) = i prod(V) prod(-P): every vertex function returns the
//     Lagrangian coefficient V (no i), every off-shell function multiplies by (-P); the propagator factor
//     "d" is passed in, already inverted, because it is helicity independent and hoisted by the generator:
//        fermion  d = -1/(q^2 - m^2 + i m Gamma)      result = d (qslash + m) (vertex)
//        vector   d = +1/(q^2 - m^2 + i m Gamma)      result = d (J - q (q.J)/m^2)   [massless: d J]
//        scalar   d = -1/(q^2 - m^2 + i m Gamma)
//     d is a real T when the line has no width, a cx<T> otherwise (template parameter D);
//   * FFV coupling (Eq. 35): L = psibar gamma^mu (gL PL + gR PR) psi V_mu, gc[0] = gL,
//     gc[1] = gR; qqg has gL = gR = -g_s with colour T^a (Eq. 36-38);
//   * template masks give the compile-time sparsity: MI / MO = which slots of the in-flowing (column) /
//     out-flowing (row) spinor are non-zero, G = which of gL, gR are non-zero.  A massless fermion line keeps
//     a single slot pair from end to end (helicity conservation), which halves the work of every FFV call.
#pragma once
#include "hg_cx.cuh"

namespace hg {

// =============================================================================== external lines
// Two-component helicity eigenstates scaled by sqrt(2|p|):  s_+ = sqrt(2|p|) chi_+ , s_- = sqrt(2|p|) chi_-
//   chi_+ = (|p|+pz, px+i py)/sqrt(2|p|(|p|+pz)),  chi_- = (-px+i py, |p|+pz)/sqrt(2|p|(|p|+pz)).
// |p|+pz is formed without cancellation for pz < 0.
template <class T>
HG_HD void helicity_basis(const Mom<T>& p, T pabs, int lam, cx<T>& s0, cx<T>& s1) {
  T pt2 = p.x * p.x + p.y * p.y;
  T ppz = hpos(p.z) ? pabs + p.z : (hpos(pabs - p.z) ? pt2 * hrcp(pabs - p.z) : T(0));
  if (!hpos(pabs)) {  // at rest: quantise along +z
    s0 = mk<T>(lam > 0 ? T(1) : T(0), T(0));
    s1 = mk<T>(lam > 0 ? T(0) : T(1), T(0));
    return;
  }
  if (!hpos(ppz)) {  // along -z
    T r = hsqrt(pabs + pabs);
    s0 = mk<T>(lam > 0 ? T(0) : -r, T(0));
    s1 = mk<T>(lam > 0 ? r : T(0), T(0));
    return;
  }
  T r = hsqrt(ppz);
  T ri = hrcp(r);
  if (lam > 0) {
    s0 = mk<T>(r, T(0));
    s1 = mk<T>(p.x * ri, p.y * ri);
  } else {
    s0 = mk<T>(-(p.x * ri), p.y * ri);
    s1 = mk<T>(r, T(0));
  }
}

// ixxxxx: flowing-IN fermion (Eq. 29).  nsf=+1: u(p,nhel/2); nsf=-1: v(p,nhel/2).
//   u(p,l) = ( sqrt(E - l|p|) chi_l ; sqrt(E + l|p|) chi_l )
//   v(p,l) = ( -l sqrt(E + l|p|) chi_-l ; l sqrt(E - l|p|) chi_-l )
template <class T>
HG_HD Sp<T> ixxxxx(const Mom<T>& p, T m, int nhel, int nsf) {
  T pabs = hsqrt(p.x * p.x + p.y * p.y + p.z * p.z);
  T rp = hsqrt(p.e + pabs);     // sqrt(E+|p|)
  T rm = m * hrcp(rp);          // sqrt(E-|p|) = m / sqrt(E+|p|)
  cx<T> s0, s1;
  int lam = nsf > 0 ? nhel : -nhel;
  helicity_basis(p, pabs, lam, s0, s1);
  // s = sqrt(2|p|) chi  ->  chi = s / sqrt(2|p|)   (at rest helicity_basis returns chi itself)
  T nrm = hpos(pabs) ? hrcp(hsqrt(pabs + pabs)) : T(1);
  T top, bot;
  if (nsf > 0) {
    top = (nhel > 0 ? rm : rp) * nrm;
    bot = (nhel > 0 ? rp : rm) * nrm;
  } else {
    top = (nhel > 0 ? -rp : rm) * nrm;   // -l sqrt(E + l|p|)
    bot = (nhel > 0 ? rm : -rp) * nrm;   //  l sqrt(E - l|p|)
  }
  Sp<T> f;
  f.c[0] = top * s0;
  f.c[1] = top * s1;
  f.c[2] = bot * s0;
  f.c[3] = bot * s1;
  return f;
}

// oxxxxx: flowing-OUT fermion (Eq. 30).  nsf=+1: ubar(p,nhel/2); nsf=-1: vbar.
// Row spinor psi^dagger gamma^0 = (conj(bottom), conj(top)).
template <class T>
HG_HD Sp<T> oxxxxx(const Mom<T>& p, T m, int nhel, int nsf) {
  Sp<T> f = ixxxxx(p, m, nhel, nsf);
  Sp<T> o;
  o.c[0] = conj(f.c[2]);
  o.c[1] = conj(f.c[3]);
  o.c[2] = conj(f.c[0]);
  o.c[3] = conj(f.c[1]);
  return o;
}

// Massless versions.  The non-zero slot pair is fixed by nhel*nsf: -1 -> slots A, +1 -> slots B (column);
// the row spinor has them swapped.  The other pair is set to zero and never read by masked callers.
template <class T>
HG_HD Sp<T> ixxxx0(const Mom<T>& p, int nhel, int nsf) {
  cx<T> s0, s1;
  int lam = nsf > 0 ? nhel : -nhel;
  helicity_basis(p, p.e, lam, s0, s1);
  Sp<T> f;
  int o = (nhel * nsf < 0) ? 0 : 2;
  f.c[2 - o] = czero<T>();
  f.c[3 - o] = czero<T>();
  if (nsf > 0) {
    f.c[o] = s0;
    f.c[o + 1] = s1;
  } else {
    f.c[o] = -s0;
    f.c[o + 1] = -s1;
  }
  return f;
}
template <class T>
HG_HD Sp<T> oxxxx0(const Mom<T>& p, int nhel, int nsf) {
  Sp<T> f = ixxxx0(p, nhel, nsf);
  Sp<T> o;
  o.c[0] = conj(f.c[2]);
  o.c[1] = conj(f.c[3]);
  o.c[2] = conj(f.c[0]);
  o.c[3] = conj(f.c[1]);
  return o;
}

// vxxxxx: vector boson (Eq. 32; body of List 5 missing, reading SURVEY.md 8c-A3):
//   eps(+-1) = (-+ e1 - i e2)/sqrt2,  e1 = d p^/d theta, e2 = d p^/(sin theta d phi);  eps(0) = (|p|, E p^)/m.
// nsv = -1 initial: eps; nsv = +1 final: conj(eps).
template <class T>
HG_HD Vc<T> vxxxxx(const Mom<T>& p, T m, int nhel, int nsv) {
  T pt2 = p.x * p.x + p.y * p.y;
  T pabs = hsqrt(pt2 + p.z * p.z);
  T pt = hsqrt(pt2);
  T ct, st, cf, sf;
  if (hpos(pabs)) {
    T ri = hrcp(pabs);
    ct = p.z * ri;
    st = pt * ri;
  } else {
    ct = T(1);
    st = T(0);
  }
  if (hpos(pt)) {
    T ri = hrcp(pt);
    cf = p.x * ri;
    sf = p.y * ri;
  } else {
    cf = T(1);
    sf = T(0);
  }
  Vc<T> v;
  if (nhel == 0) {
    T mi = hrcp(m);
    T em = p.e * mi;
    v.c[0] = mk<T>(pabs * mi, T(0));
    v.c[1] = mk<T>(em * st * cf, T(0));
    v.c[2] = mk<T>(em * st * sf, T(0));
    v.c[3] = mk<T>(em * ct, T(0));
    return v;
  }
  const T rs2 = T(0.70710678118654752440);
  T l = nhel > 0 ? -rs2 : rs2;          // -lambda/sqrt2
  T s = nsv > 0 ? rs2 : -rs2;           // imaginary part: -1/sqrt2 (initial), +1/sqrt2 (final, conjugated)
  v.c[0] = czero<T>();
  v.c[1] = mk<T>(l * ct * cf, -(s * sf));
  v.c[2] = mk<T>(l * ct * sf, s * cf);
  v.c[3] = mk<T>(-(l * st), T(0));
  return v;
}
// eps(-lambda) = -conj(eps(lambda)) for lambda = +-1 (both for nsv = +-1).
template <class T>
HG_HD Vc<T> vflip(const Vc<T>& v) {
  Vc<T> r;
  for (int i = 0; i < 4; ++i) r.c[i] = mk<T>(-v.c[i].re, v.c[i].im);
  return r;
}

// sxxxxx: scalar boson (Eq. 34; List 6 PAPER.md:1537-1549): the wavefunction is 1.
template <class T>
HG_HD cx<T> sxxxxx() {
  return mk<T>(T(1), T(0));
}

// =============================================================================== 2x2 blocks
// M_S(k) = k0 + S k.sigma for a real momentum k, acting on a column (y = M w) or a row (y = r M).
template <int S, class T>
HG_HD void sig_col(const Mom<T>& k, cx<T> w0, cx<T> w1, cx<T>& y0, cx<T>& y1) {
  T a = S > 0 ? k.e + k.z : k.e - k.z;
  T b = S > 0 ? k.e - k.z : k.e + k.z;
  T x = S > 0 ? k.x : -k.x;
  T y = S > 0 ? k.y : -k.y;
  y0 = mk<T>(a * w0.re + x * w1.re + y * w1.im, a * w0.im + x * w1.im - y * w1.re);
  y1 = mk<T>(b * w1.re + x * w0.re - y * w0.im, b * w1.im + x * w0.im + y * w0.re);
}
template <int S, class T>
HG_HD void sig_row(const Mom<T>& k, cx<T> r0, cx<T> r1, cx<T>& y0, cx<T>& y1) {
  T a = S > 0 ? k.e + k.z : k.e - k.z;
  T b = S > 0 ? k.e - k.z : k.e + k.z;
  T x = S > 0 ? k.x : -k.x;
  T y = S > 0 ? k.y : -k.y;
  y0 = mk<T>(a * r0.re + x * r1.re - y * r1.im, a * r0.im + x * r1.im + y * r1.re);
  y1 = mk<T>(b * r1.re + x * r0.re + y * r0.im, b * r1.im + x * r0.im - y * r0.re);
}
// Same for a complex vector V.
template <int S, class T>
HG_HD void sig_col(const Vc<T>& v, cx<T> w0, cx<T> w1, cx<T>& y0, cx<T>& y1) {
  cx<T> a = S > 0 ? v.c[0] + v.c[3] : v.c[0] - v.c[3];
  cx<T> b = S > 0 ? v.c[0] - v.c[3] : v.c[0] + v.c[3];
  cx<T> ur = mk<T>(v.c[1].re + v.c[2].im, v.c[1].im - v.c[2].re);  // V1 - i V2
  cx<T> ll = mk<T>(v.c[1].re - v.c[2].im, v.c[1].im + v.c[2].re);  // V1 + i V2
  if (S > 0) {
    y0 = cfma(ur, w1, a * w0);
    y1 = cfma(ll, w0, b * w1);
  } else {
    y0 = a * w0 - ur * w1;
    y1 = b * w1 - ll * w0;
  }
}
template <int S, class T>
HG_HD void sig_row(const Vc<T>& v, cx<T> r0, cx<T> r1, cx<T>& y0, cx<T>& y1) {
  cx<T> a = S > 0 ? v.c[0] + v.c[3] : v.c[0] - v.c[3];
  cx<T> b = S > 0 ? v.c[0] - v.c[3] : v.c[0] + v.c[3];
  cx<T> ur = mk<T>(v.c[1].re + v.c[2].im, v.c[1].im - v.c[2].re);
  cx<T> ll = mk<T>(v.c[1].re - v.c[2].im, v.c[1].im + v.c[2].re);
  if (S > 0) {
    y0 = cfma(r1, ll, r0 * a);
    y1 = cfma(r0, ur, r1 * b);
  } else {
    y0 = r0 * a - r1 * ll;
    y1 = r1 * b - r0 * ur;
  }
}

// Polarisation vector of a massless vector leg in light-cone form: eps^0 = 0 and eps^3 is real (vxxxxx), so
// M_+-(eps) = +-[[eps3, V1 - i V2], [V1 + i V2, -eps3]] needs no additions and two real x complex products.
template <class T>
struct Pol {
  T v3;
  cx<T> ur, ll;   // V1 - i V2, V1 + i V2
};
template <class T>
HG_HD Pol<T> to_pol(const Vc<T>& v) {
  Pol<T> p;
  p.v3 = v.c[3].re;
  p.ur = mk<T>(v.c[1].re + v.c[2].im, v.c[1].im - v.c[2].re);
  p.ll = mk<T>(v.c[1].re - v.c[2].im, v.c[1].im + v.c[2].re);
  return p;
}
template <int S, class T>
HG_HD void sig_col(const Pol<T>& v, cx<T> w0, cx<T> w1, cx<T>& y0, cx<T>& y1) {
  const cx<T> a = cfma(v.ur, w1, v.v3 * w0);          // eps3 w0 + (V1 - i V2) w1
  const cx<T> b = cfma(v.ll, w0, (-v.v3) * w1);       // (V1 + i V2) w0 - eps3 w1
  y0 = S > 0 ? a : -a;
  y1 = S > 0 ? b : -b;
}
template <int S, class T>
HG_HD void sig_row(const Pol<T>& v, cx<T> r0, cx<T> r1, cx<T>& y0, cx<T>& y1) {
  const cx<T> a = cfma(r1, v.ll, v.v3 * r0);          // r0 eps3 + r1 (V1 + i V2)
  const cx<T> b = cfma(r0, v.ur, (-v.v3) * r1);       // r0 (V1 - i V2) - r1 eps3
  y0 = S > 0 ? a : -a;
  y1 = S > 0 ? b : -b;
}

// =============================================================================== FFV (Eq. 35)
// iovxxx: amplitude  <fo| gamma^mu (gL PL + gR PR) |fi> V_mu
//   = gL foB (V0 + V.sigma) fiA + gR foA (V0 - V.sigma) fiB
template <int MI, int MO, int G, class T>
HG_HD cx<T> iovxxx(const Sp<T>& fi, const Sp<T>& fo, const Vc<T>& v, T gL, T gR) {
  cx<T> r = czero<T>();
  if ((MI & SLOT_A) && (MO & SLOT_B) && (G & CPL_L)) {
    cx<T> y0, y1;
    sig_col<+1>(v, fi.c[0], fi.c[1], y0, y1);
    r = gL * cfma(fo.c[3], y1, fo.c[2] * y0);
  }
  if ((MI & SLOT_B) && (MO & SLOT_A) && (G & CPL_R)) {
    cx<T> y0, y1;
    sig_col<-1>(v, fi.c[2], fi.c[3], y0, y1);
    r = r + gR * cfma(fo.c[1], y1, fo.c[0] * y0);
  }
  return r;
}

// fvixxx: off-shell flowing-IN fermion  d (qslash + m) Vslash (gL PL + gR PR) |fi>
// q = momentum along the fermion arrow (= sum of incoming momenta of the subtree), d = -1/(q^2-m^2+i m G).
template <int MI, int G, bool MASSIVE, class T, class D, class V>
HG_HD Sp<T> fvixxx(const Sp<T>& fi, const V& v, T gL, T gR, const Mom<T>& q, T m, D d) {
  constexpr bool L = (MI & SLOT_A) && (G & CPL_L);  // w_B = gL M+(V) fi_A
  constexpr bool R = (MI & SLOT_B) && (G & CPL_R);  // w_A = gR M-(V) fi_B
  if constexpr (!MASSIVE && (L != R)) {
    // one chirality on a massless line: coupling and propagator factor are applied once, at the end
    Sp<T> f;
    for (int i = 0; i < 4; ++i) f.c[i] = czero<T>();
    cx<T> w0, w1, y0, y1;
    const D gd = (L ? gL : gR) * d;
    if (L) {
      sig_col<+1>(v, fi.c[0], fi.c[1], w0, w1);
      sig_col<-1>(q, w0, w1, y0, y1);
      f.c[0] = gd * y0;
      f.c[1] = gd * y1;
    } else {
      sig_col<-1>(v, fi.c[2], fi.c[3], w0, w1);
      sig_col<+1>(q, w0, w1, y0, y1);
      f.c[2] = gd * y0;
      f.c[3] = gd * y1;
    }
    return f;
  }
  cx<T> wB0 = czero<T>(), wB1 = czero<T>(), wA0 = czero<T>(), wA1 = czero<T>();
  if (L) {
    sig_col<+1>(v, fi.c[0], fi.c[1], wB0, wB1);
    wB0 = gL * wB0;
    wB1 = gL * wB1;
  }
  if (R) {
    sig_col<-1>(v, fi.c[2], fi.c[3], wA0, wA1);
    wA0 = gR * wA0;
    wA1 = gR * wA1;
  }
  Sp<T> f;
  for (int i = 0; i < 4; ++i) f.c[i] = czero<T>();
  // (qslash + m) w :  A <- M-(q) w_B + m w_A ,  B <- M+(q) w_A + m w_B
  if (L || (R && MASSIVE)) {
    cx<T> y0 = czero<T>(), y1 = czero<T>();
    if (L) sig_col<-1>(q, wB0, wB1, y0, y1);
    if (R && MASSIVE) {
      y0 = y0 + m * wA0;
      y1 = y1 + m * wA1;
    }
    f.c[0] = d * y0;
    f.c[1] = d * y1;
  }
  if (R || (L && MASSIVE)) {
    cx<T> y0 = czero<T>(), y1 = czero<T>();
    if (R) sig_col<+1>(q, wA0, wA1, y0, y1);
    if (L && MASSIVE) {
      y0 = y0 + m * wB0;
      y1 = y1 + m * wB1;
    }
    f.c[2] = d * y0;
    f.c[3] = d * y1;
  }
  return f;
}

// fvoxxx: off-shell flowing-OUT fermion  d <fo| Vslash (gL PL + gR PR) (qslash + m)
// q = momentum along the fermion arrow (= MINUS the sum of incoming momenta of the subtree).
template <int MO, int G, bool MASSIVE, class T, class D, class V>
HG_HD Sp<T> fvoxxx(const Sp<T>& fo, const V& v, T gL, T gR, const Mom<T>& q, T m, D d) {
  constexpr bool L = (MO & SLOT_B) && (G & CPL_L);  // w_A = gL fo_B M+(V)
  constexpr bool R = (MO & SLOT_A) && (G & CPL_R);  // w_B = gR fo_A M-(V)
  if constexpr (!MASSIVE && (L != R)) {
    Sp<T> f;
    for (int i = 0; i < 4; ++i) f.c[i] = czero<T>();
    cx<T> w0, w1, y0, y1;
    const D gd = (L ? gL : gR) * d;
    if (L) {
      sig_row<+1>(v, fo.c[2], fo.c[3], w0, w1);
      sig_row<-1>(q, w0, w1, y0, y1);
      f.c[2] = gd * y0;
      f.c[3] = gd * y1;
    } else {
      sig_row<-1>(v, fo.c[0], fo.c[1], w0, w1);
      sig_row<+1>(q, w0, w1, y0, y1);
      f.c[0] = gd * y0;
      f.c[1] = gd * y1;
    }
    return f;
  }
  cx<T> wA0 = czero<T>(), wA1 = czero<T>(), wB0 = czero<T>(), wB1 = czero<T>();
  if (L) {
    sig_row<+1>(v, fo.c[2], fo.c[3], wA0, wA1);
    wA0 = gL * wA0;
    wA1 = gL * wA1;
  }
  if (R) {
    sig_row<-1>(v, fo.c[0], fo.c[1], wB0, wB1);
    wB0 = gR * wB0;
    wB1 = gR * wB1;
  }
  Sp<T> f;
  for (int i = 0; i < 4; ++i) f.c[i] = czero<T>();
  // w (qslash + m) :  A <- w_B M+(q) + m w_A ,  B <- w_A M-(q) + m w_B
  if (R || (L && MASSIVE)) {
    cx<T> y0 = czero<T>(), y1 = czero<T>();
    if (R) sig_row<+1>(q, wB0, wB1, y0, y1);
    if (L && MASSIVE) {
      y0 = y0 + m * wA0;
      y1 = y1 + m * wA1;
    }
    f.c[0] = d * y0;
    f.c[1] = d * y1;
  }
  if (L || (R && MASSIVE)) {
    cx<T> y0 = czero<T>(), y1 = czero<T>();
    if (L) sig_row<-1>(q, wA0, wA1, y0, y1);
    if (R && MASSIVE) {
      y0 = y0 + m * wB0;
      y1 = y1 + m * wB1;
    }
    f.c[2] = d * y0;
    f.c[3] = d * y1;
  }
  return f;
}

// =============================================================================== massless single-chirality lines
// On a massless fermion line with one chirality the off-shell spinor is  (g d) M_-+(q) M_+-(V) w : the generator
// folds the coupling g and the (real) propagator factor d into the momentum ONCE per event and stores it in
// light-cone components,  kq = g d (q0 + q3, q1, q2, q0 - q3)  kept in a Mom<T> as (e, x, y, z)  (lc_scaled), so the
// second matrix product needs neither the two additions q0 +- q3 nor the final scaling: 12 instead of 18 fp64
// instructions, and one staged word less per line (emit.py "scaled momenta").
template <class T>
HG_HD Mom<T> lc_scaled(const Mom<T>& q, T s) {
  return mkmom<T>(s * (q.e + q.z), s * q.x, s * q.y, s * (q.e - q.z));
}
// M_S(q) w for q in light-cone components: M_+ = [[a, x - i y], [x + i y, b]], M_- = [[b, -(x - i y)], [-(x + i y), a]]
template <int S, class T>
HG_HD void lc_col(const Mom<T>& k, cx<T> w0, cx<T> w1, cx<T>& y0, cx<T>& y1) {
  if (S > 0) {
    y0 = mk<T>(k.e * w0.re + k.x * w1.re + k.y * w1.im, k.e * w0.im + k.x * w1.im - k.y * w1.re);
    y1 = mk<T>(k.z * w1.re + k.x * w0.re - k.y * w0.im, k.z * w1.im + k.x * w0.im + k.y * w0.re);
  } else {
    y0 = mk<T>(k.z * w0.re - k.x * w1.re - k.y * w1.im, k.z * w0.im - k.x * w1.im + k.y * w1.re);
    y1 = mk<T>(k.e * w1.re - k.x * w0.re + k.y * w0.im, k.e * w1.im - k.x * w0.im - k.y * w0.re);
  }
}
template <int S, class T>
HG_HD void lc_row(const Mom<T>& k, cx<T> r0, cx<T> r1, cx<T>& y0, cx<T>& y1) {
  if (S > 0) {
    y0 = mk<T>(k.e * r0.re + k.x * r1.re - k.y * r1.im, k.e * r0.im + k.x * r1.im + k.y * r1.re);
    y1 = mk<T>(k.z * r1.re + k.x * r0.re + k.y * r0.im, k.z * r1.im + k.x * r0.im - k.y * r0.re);
  } else {
    y0 = mk<T>(k.z * r0.re - k.x * r1.re + k.y * r1.im, k.z * r0.im - k.x * r1.im - k.y * r1.re);
    y1 = mk<T>(k.e * r1.re - k.x * r0.re - k.y * r0.im, k.e * r1.im - k.x * r0.im + k.y * r0.re);
  }
}
// fvixxx / fvoxxx of a massless single-chirality line with the scaled light-cone momentum kq = lc_scaled(q, g d)
// (fvoxx0: q = MINUS the sum of incoming momenta, as for fvoxxx)
template <int MI, int G, class T, class V>
HG_HD Sp<T> fvixx0(const Sp<T>& fi, const V& v, const Mom<T>& kq) {
  constexpr bool L = (MI & SLOT_A) && (G & CPL_L);
  constexpr bool R = (MI & SLOT_B) && (G & CPL_R);
  static_assert(L != R, "single chirality only");
  Sp<T> f;
  for (int i = 0; i < 4; ++i) f.c[i] = czero<T>();
  cx<T> w0, w1;
  if (L) {
    sig_col<+1>(v, fi.c[0], fi.c[1], w0, w1);
    lc_col<-1>(kq, w0, w1, f.c[0], f.c[1]);
  } else {
    sig_col<-1>(v, fi.c[2], fi.c[3], w0, w1);
    lc_col<+1>(kq, w0, w1, f.c[2], f.c[3]);
  }
  return f;
}
template <int MO, int G, class T, class V>
HG_HD Sp<T> fvoxx0(const Sp<T>& fo, const V& v, const Mom<T>& kq) {
  constexpr bool L = (MO & SLOT_B) && (G & CPL_L);
  constexpr bool R = (MO & SLOT_A) && (G & CPL_R);
  static_assert(L != R, "single chirality only");
  Sp<T> f;
  for (int i = 0; i < 4; ++i) f.c[i] = czero<T>();
  cx<T> w0, w1;
  if (L) {
    sig_row<+1>(v, fo.c[2], fo.c[3], w0, w1);
    lc_row<-1>(kq, w0, w1, f.c[2], f.c[3]);
  } else {
    sig_row<-1>(v, fo.c[0], fo.c[1], w0, w1);
    lc_row<+1>(kq, w0, w1, f.c[0], f.c[1]);
  }
  return f;
}

// the same with the result rescaled by r = (coupling of this vertex) / (coupling folded into kq)
template <int MI, int G, class T, class V>
HG_HD Sp<T> fvixx0s(const Sp<T>& fi, const V& v, const Mom<T>& kq, T r) {
  Sp<T> f = fvixx0<MI, G>(fi, v, kq);
  for (int i = 0; i < 4; ++i) f.c[i] = r * f.c[i];
  return f;
}
template <int MO, int G, class T, class V>
HG_HD Sp<T> fvoxx0s(const Sp<T>& fo, const V& v, const Mom<T>& kq, T r) {
  Sp<T> f = fvoxx0<MO, G>(fo, v, kq);
  for (int i = 0; i < 4; ++i) f.c[i] = r * f.c[i];
  return f;
}

// Bare FFV current  J^mu = <fo| gamma^mu (gL PL + gR PR) |fi>  (upper index):
//   J^0 = gL foB.fiA + gR foA.fiB ,  J^i = -gL foB sigma^i fiA + gR foA sigma^i fiB
template <int MI, int MO, int G, class T>
HG_HD Vc<T> ffv_current(const Sp<T>& fi, const Sp<T>& fo, T gL, T gR) {
  Vc<T> j;
  for (int i = 0; i < 4; ++i) j.c[i] = czero<T>();
  if ((MI & SLOT_A) && (MO & SLOT_B) && (G & CPL_L)) {
    cx<T> r0 = gL * fo.c[2], r1 = gL * fo.c[3];
    cx<T> a = r0 * fi.c[0], b = r1 * fi.c[1], c = r0 * fi.c[1], e = r1 * fi.c[0];
    j.c[0] = a + b;
    j.c[3] = b - a;                  // -(r0 c0 - r1 c1)
    j.c[1] = -(c + e);               // -(r0 c1 + r1 c0)
    j.c[2] = times_i(c - e);         // -i (r1 c0 - r0 c1)
  }
  if ((MI & SLOT_B) && (MO & SLOT_A) && (G & CPL_R)) {
    cx<T> r0 = gR * fo.c[0], r1 = gR * fo.c[1];
    cx<T> a = r0 * fi.c[2], b = r1 * fi.c[3], c = r0 * fi.c[3], e = r1 * fi.c[2];
    j.c[0] = j.c[0] + (a + b);
    j.c[3] = j.c[3] + (a - b);
    j.c[1] = j.c[1] + (c + e);
    j.c[2] = j.c[2] + times_i(e - c);
  }
  return j;
}

// Vector propagator applied to a bare current: massless / Feynman gauge d J; massive / unitary gauge
// d (J - q (q.J) / m^2)   (reading A4: real m^2 in the q q / m^2 term).
template <bool UNITARY, class T, class D, class R>
HG_HD Vc<T> vprop(const Vc<T>& j, const Mom<T>& q, R rm2, D d) {
  Vc<T> w;
  if (UNITARY) {
    cx<T> s = rm2 * vdot(q, j);
    w.c[0] = d * (j.c[0] - q.e * s);
    w.c[1] = d * (j.c[1] - q.x * s);
    w.c[2] = d * (j.c[2] - q.y * s);
    w.c[3] = d * (j.c[3] - q.z * s);
  } else {
    for (int i = 0; i < 4; ++i) w.c[i] = d * j.c[i];
  }
  return w;
}

// jioxxx: off-shell vector from a fermion pair.  q = total momentum, rm2 = 1/m^2.
template <int MI, int MO, int G, bool UNITARY, class T, class D, class R>
HG_HD Vc<T> jioxxx(const Sp<T>& fi, const Sp<T>& fo, T gL, T gR, const Mom<T>& q, R rm2, D d) {
  return vprop<UNITARY>(ffv_current<MI, MO, G>(fi, fo, gL, gR), q, rm2, d);
}

// massless vector line (Feynman gauge): d J, no momentum needed
template <int MI, int MO, int G, class T, class D>
HG_HD Vc<T> jioxx0(const Sp<T>& fi, const Sp<T>& fo, T gL, T gR, D d) {
  // the current is linear in the couplings: the (real) propagator factor is folded into the ones in use
  const bool l = (MI & SLOT_A) && (MO & SLOT_B) && (G & CPL_L), r = (MI & SLOT_B) && (MO & SLOT_A) && (G & CPL_R);
  return ffv_current<MI, MO, G>(fi, fo, l ? gL * d : gL, r ? gR * d : gR);
}

// =============================================================================== VVV (Eq. 40-44)
// vvvxxx: g [ (v1.v2)(k1-k2).v3 + (v2.v3)(k2-k3).v1 + (v3.v1)(k3-k1).v2 ], all momenta incoming
// (PAPER.md:535-567, 1773-1810).  For gluons the colour factor i f^{abc} is handled by the generator.
template <class T>
HG_HD cx<T> vvvxxx(const Vc<T>& v1, const Vc<T>& v2, const Vc<T>& v3, T g, const Mom<T>& k1,
                   const Mom<T>& k2, const Mom<T>& k3) {
  cx<T> r = vdot(v1, v2) * vdot(k1 - k2, v3);
  r = cfma(vdot(v2, v3), vdot(k2 - k3, v1), r);
  r = cfma(vdot(v3, v1), vdot(k3 - k1, v2), r);
  return g * r;
}
// jvvxxx: off-shell vector from two vectors; k3 = -(k1+k2).
//   J = g [ (v1.v2)(k1-k2) + v2 ((2 k2 + k1).v1) - v1 ((2 k1 + k2).v2) ],  result = vprop(J, k1+k2)
template <bool UNITARY, class T, class D, class R>
HG_HD Vc<T> jvvxxx(const Vc<T>& v1, const Vc<T>& v2, T g, const Mom<T>& k1, const Mom<T>& k2, R rm2, D d) {
  cx<T> d12 = g * vdot(v1, v2);
  cx<T> a = g * vdot(k2 + k2 + k1, v1);
  cx<T> b = g * vdot(k1 + k1 + k2, v2);
  Mom<T> dk = k1 - k2;
  Vc<T> j;
  j.c[0] = cfma(a, v2.c[0], dk.e * d12) - b * v1.c[0];
  j.c[1] = cfma(a, v2.c[1], dk.x * d12) - b * v1.c[1];
  j.c[2] = cfma(a, v2.c[2], dk.y * d12) - b * v1.c[2];
  j.c[3] = cfma(a, v2.c[3], dk.z * d12) - b * v1.c[3];
  return vprop<UNITARY>(j, k1 + k2, rm2, d);
}

// =============================================================================== VVVV (Eq. 47-49)
// ggggxx: one colour structure of the four-gluon vertex, g2 [ (v1.v3)(v2.v4) - (v2.v3)(v1.v4) ], which
// multiplies the colour factor (i f^{12e})(i f^{34e}); the other two structures are the calls with
// (1,3,2,4) and (2,3,1,4)-type argument permutations (C.44-C.48).
template <class T>
HG_HD cx<T> ggggxx(const Vc<T>& v1, const Vc<T>& v2, const Vc<T>& v3, const Vc<T>& v4, T g2) {
  cx<T> r = vdot(v1, v3) * vdot(v2, v4) - vdot(v2, v3) * vdot(v1, v4);
  return g2 * r;
}
// jgggxx: off-shell gluon, same structure:  d g2 [ (v1.v3) v2 - (v2.v3) v1 ]   (C.49-C.52)
template <class T, class D>
HG_HD Vc<T> jgggxx(const Vc<T>& v1, const Vc<T>& v2, const Vc<T>& v3, T g2, D d) {
  cx<T> a = g2 * vdot(v1, v3);
  cx<T> b = g2 * vdot(v2, v3);
  Vc<T> w;
  for (int i = 0; i < 4; ++i) w.c[i] = d * (a * v2.c[i] - b * v1.c[i]);
  return w;
}

// =============================================================================== closing on a massless vector leg
// The amplitude of a diagram is linear in the wavefunction of its last external leg.  When that leg is a massless
// vector boson, eps(h) = (0, s Re e + i Im e) with e = eps(+1), s = +1 (h = +1) or -1 (h = -1, vflip), so
//   amplitude(h) = eps(h).B = -(s rb + i ib),   rb = sum_i Re(e_i) B_i,  ib = sum_i Im(e_i) B_i   (i = 1..3)
// for the bare current B of the closing vertex (the off-shell functions below without their propagator).  The
// generator accumulates rb, ib per colour flow once and forms both helicities at the end: the loop over the last
// helicity and half of the closing arithmetic disappear.
template <class T>
HG_HD void close_proj(const Vc<T>& e, const Vc<T>& b, cx<T>& rb, cx<T>& ib) {
  rb = mk<T>(e.c[1].re * b.c[1].re + e.c[2].re * b.c[2].re + e.c[3].re * b.c[3].re,
             e.c[1].re * b.c[1].im + e.c[2].re * b.c[2].im + e.c[3].re * b.c[3].im);
  ib = mk<T>(e.c[1].im * b.c[1].re + e.c[2].im * b.c[2].re + e.c[3].im * b.c[3].re,
             e.c[1].im * b.c[1].im + e.c[2].im * b.c[2].im + e.c[3].im * b.c[3].im);
}
// Closing an FFV vertex on the massless vector leg through a DRESSED spinor.  rb = sum_i x_i J_i (i = 1..3) with
// J = ffv_current(fi, fo) and x = Re eps(+1) (PART = 0) or Im eps(+1) (PART = 1; its third component vanishes) is
// bilinear in the two spinors:  rb = D . fi  with the row spinor D = <fo| x_i gamma^i (gL PL + gR PR), or
// rb = fo . C  with the column spinor C.  When one of the spinors lives outside the helicity loops the generator
// dresses it once per event (dress_row / dress_col) and every closing inside the loops is a plain spinor dot
// product (sdot): 2 complex FMAs per chirality instead of the current + projection (gen/emit.py "closing by spinor").
//   L part (fo slots B, fi slots A):  J_1 = -gL (r0 c1 + r1 c0), J_2 = i gL (r0 c1 - r1 c0), J_3 = gL (r1 c1 - r0 c0)
//   R part (fo slots A, fi slots B):  J_1 =  gR (r0 c1 + r1 c0), J_2 = i gR (r1 c0 - r0 c1), J_3 = gR (r0 c0 - r1 c1)
template <int PART, class T>
HG_HD void dress_pair(const Vc<T>& e, T g, cx<T> s0, cx<T> s1, bool row, bool left, cx<T>& d0, cx<T>& d1) {
  const T x1 = PART ? e.c[1].im : e.c[1].re, x2 = PART ? e.c[2].im : e.c[2].re;
  // (x1 + i x2) and (x1 - i x2): a dressed row has the "+" one in d0, a dressed column the "-" one
  const bool plus_first = row;
  const cx<T> p = mk<T>(x1, plus_first ? x2 : -x2), m = mk<T>(x1, plus_first ? -x2 : x2);
  cx<T> a = p * s1, b = m * s0;
  if (PART == 0) {
    const T x3 = e.c[3].re;
    a = a + x3 * s0;
    b = b - x3 * s1;
  }
  // L part: d0 = -g (x3 s0 + p s1), d1 = g (x3 s1 - m s0);  R part: the opposite sign
  const T gs = left ? -g : g;
  d0 = gs * a;
  d1 = gs * b;
}
template <int MO, int G, int PART, class T>
HG_HD Sp<T> dress_row(const Sp<T>& fo, const Vc<T>& e, T gL, T gR) {
  Sp<T> d;
  for (int i = 0; i < 4; ++i) d.c[i] = czero<T>();
  if ((MO & SLOT_B) && (G & CPL_L)) dress_pair<PART>(e, gL, fo.c[2], fo.c[3], true, true, d.c[0], d.c[1]);
  if ((MO & SLOT_A) && (G & CPL_R)) dress_pair<PART>(e, gR, fo.c[0], fo.c[1], true, false, d.c[2], d.c[3]);
  return d;
}
template <int MI, int G, int PART, class T>
HG_HD Sp<T> dress_col(const Sp<T>& fi, const Vc<T>& e, T gL, T gR) {
  Sp<T> d;
  for (int i = 0; i < 4; ++i) d.c[i] = czero<T>();
  if ((MI & SLOT_A) && (G & CPL_L)) dress_pair<PART>(e, gL, fi.c[0], fi.c[1], false, true, d.c[2], d.c[3]);
  if ((MI & SLOT_B) && (G & CPL_R)) dress_pair<PART>(e, gR, fi.c[2], fi.c[3], false, false, d.c[0], d.c[1]);
  return d;
}
// plain (unconjugated) dot product of two spinors over the slot pairs of mask M
template <int M, class T>
HG_HD cx<T> sdot(const Sp<T>& a, const Sp<T>& b) {
  cx<T> r = czero<T>();
  if (M & SLOT_A) r = cfma(a.c[1], b.c[1], a.c[0] * b.c[0]);
  if (M & SLOT_B) {
    if (M & SLOT_A)
      r = cfma(a.c[3], b.c[3], cfma(a.c[2], b.c[2], r));
    else
      r = cfma(a.c[3], b.c[3], a.c[2] * b.c[2]);
  }
  return r;
}
// amplitude for helicity sign s from the accumulated projections
template <class T>
HG_HD cx<T> close_amp(cx<T> x, cx<T> y, T s) {
  return mk<T>(y.im - s * x.re, -(s * x.im) - y.re);
}
// bare three-vector current (jvvxxx without propagator):  v3.jvv_bare(v1,v2) = vvvxxx(v1,v2,v3), k3 = -(k1+k2)
template <class T>
HG_HD Vc<T> jvv_bare(const Vc<T>& v1, const Vc<T>& v2, T g, const Mom<T>& k1, const Mom<T>& k2) {
  cx<T> d12 = g * vdot(v1, v2);
  cx<T> a = g * vdot(k2 + k2 + k1, v1);
  cx<T> b = g * vdot(k1 + k1 + k2, v2);
  Mom<T> dk = k1 - k2;
  Vc<T> j;
  j.c[0] = cfma(a, v2.c[0], dk.e * d12) - b * v1.c[0];
  j.c[1] = cfma(a, v2.c[1], dk.x * d12) - b * v1.c[1];
  j.c[2] = cfma(a, v2.c[2], dk.y * d12) - b * v1.c[2];
  j.c[3] = cfma(a, v2.c[3], dk.z * d12) - b * v1.c[3];
  return j;
}
// bare four-gluon current of one colour structure:  v4.jggg_bare(v1,v2,v3) = ggggxx(v1,v2,v3,v4)
template <class T>
HG_HD Vc<T> jggg_bare(const Vc<T>& v1, const Vc<T>& v2, const Vc<T>& v3, T g2) {
  cx<T> a = g2 * vdot(v1, v3);
  cx<T> b = g2 * vdot(v2, v3);
  Vc<T> w;
  for (int i = 0; i < 4; ++i) w.c[i] = a * v2.c[i] - b * v1.c[i];
  return w;
}

// =============================================================================== FFS (Eq. 39)
// L = psibar (gL PL + gR PR) psi S.  In the chiral basis PL keeps column slots A and pairs them with ROW slots A
// (psibar = psi^dagger gamma^0 has the conjugate RIGHT part in its slots A), PR pairs slots B with B.
// iosxxx: amplitude (C.4.1)
template <int MI, int MO, int G, class T, class C_>
HG_HD cx<T> iosxxx(const Sp<T>& fi, const Sp<T>& fo, cx<T> s, C_ gL, C_ gR) {
  cx<T> r = czero<T>();
  if ((MI & SLOT_A) && (MO & SLOT_A) && (G & CPL_L)) r = gL * cfma(fo.c[1], fi.c[1], fo.c[0] * fi.c[0]);
  if ((MI & SLOT_B) && (MO & SLOT_B) && (G & CPL_R)) r = r + gR * cfma(fo.c[3], fi.c[3], fo.c[2] * fi.c[2]);
  return s * r;
}
// hioxxx: off-shell scalar from a fermion pair (C.4.4); d = -1/(q^2 - m^2 + i m Gamma)
template <int MI, int MO, int G, class T, class D, class C_>
HG_HD cx<T> hioxxx(const Sp<T>& fi, const Sp<T>& fo, C_ gL, C_ gR, D d) {
  cx<T> r = czero<T>();
  if ((MI & SLOT_A) && (MO & SLOT_A) && (G & CPL_L)) r = gL * cfma(fo.c[1], fi.c[1], fo.c[0] * fi.c[0]);
  if ((MI & SLOT_B) && (MO & SLOT_B) && (G & CPL_R)) r = r + gR * cfma(fo.c[3], fi.c[3], fo.c[2] * fi.c[2]);
  return d * r;
}
// fsixxx: off-shell flowing-IN fermion  d (qslash + m) (gL PL + gR PR) |fi> S   (C.4.2)
template <int MI, int G, bool MASSIVE, class T, class D, class C_>
HG_HD Sp<T> fsixxx(const Sp<T>& fi, cx<T> s, C_ gL, C_ gR, const Mom<T>& q, T m, D d) {
  constexpr bool L = (MI & SLOT_A) && (G & CPL_L);  // w_A = gL S fi_A
  constexpr bool R = (MI & SLOT_B) && (G & CPL_R);  // w_B = gR S fi_B
  cx<T> wA0 = czero<T>(), wA1 = czero<T>(), wB0 = czero<T>(), wB1 = czero<T>();
  if (L) {
    const cx<T> g = gL * s;
    wA0 = g * fi.c[0];
    wA1 = g * fi.c[1];
  }
  if (R) {
    const cx<T> g = gR * s;
    wB0 = g * fi.c[2];
    wB1 = g * fi.c[3];
  }
  Sp<T> f;
  for (int i = 0; i < 4; ++i) f.c[i] = czero<T>();
  // (qslash + m) w :  A <- M-(q) w_B + m w_A ,  B <- M+(q) w_A + m w_B
  if (R || (L && MASSIVE)) {
    cx<T> y0 = czero<T>(), y1 = czero<T>();
    if (R) sig_col<-1>(q, wB0, wB1, y0, y1);
    if (L && MASSIVE) {
      y0 = y0 + m * wA0;
      y1 = y1 + m * wA1;
    }
    f.c[0] = d * y0;
    f.c[1] = d * y1;
  }
  if (L || (R && MASSIVE)) {
    cx<T> y0 = czero<T>(), y1 = czero<T>();
    if (L) sig_col<+1>(q, wA0, wA1, y0, y1);
    if (R && MASSIVE) {
      y0 = y0 + m * wB0;
      y1 = y1 + m * wB1;
    }
    f.c[2] = d * y0;
    f.c[3] = d * y1;
  }
  return f;
}
// fsoxxx: off-shell flowing-OUT fermion  d <fo| (gL PL + gR PR) S (qslash + m)   (C.4.3)
template <int MO, int G, bool MASSIVE, class T, class D, class C_>
HG_HD Sp<T> fsoxxx(const Sp<T>& fo, cx<T> s, C_ gL, C_ gR, const Mom<T>& q, T m, D d) {
  constexpr bool L = (MO & SLOT_A) && (G & CPL_L);  // w_A = gL S fo_A
  constexpr bool R = (MO & SLOT_B) && (G & CPL_R);  // w_B = gR S fo_B
  cx<T> wA0 = czero<T>(), wA1 = czero<T>(), wB0 = czero<T>(), wB1 = czero<T>();
  if (L) {
    const cx<T> g = gL * s;
    wA0 = g * fo.c[0];
    wA1 = g * fo.c[1];
  }
  if (R) {
    const cx<T> g = gR * s;
    wB0 = g * fo.c[2];
    wB1 = g * fo.c[3];
  }
  Sp<T> f;
  for (int i = 0; i < 4; ++i) f.c[i] = czero<T>();
  // w (qslash + m) :  A <- w_B M+(q) + m w_A ,  B <- w_A M-(q) + m w_B
  if (R || (L && MASSIVE)) {
    cx<T> y0 = czero<T>(), y1 = czero<T>();
    if (R) sig_row<+1>(q, wB0, wB1, y0, y1);
    if (L && MASSIVE) {
      y0 = y0 + m * wA0;
      y1 = y1 + m * wA1;
    }
    f.c[0] = d * y0;
    f.c[1] = d * y1;
  }
  if (L || (R && MASSIVE)) {
    cx<T> y0 = czero<T>(), y1 = czero<T>();
    if (L) sig_row<-1>(q, wA0, wA1, y0, y1);
    if (R && MASSIVE) {
      y0 = y0 + m * wB0;
      y1 = y1 + m * wB1;
    }
    f.c[2] = d * y0;
    f.c[3] = d * y1;
  }
  return f;
}

// =============================================================================== VVS, VVSS, SSS (Eq. 50-52)
// L_VVS = g (V1.V2) S, L_VVSS = g (V1.V2) S3 S4, L_SSS = g S1 S2 S3 (C.7-C.9); g is the
// coefficient of the Feynman rule (W W H: gW mW, Z Z H: gZ mZ, W W H H: gW^2/2, Z Z H H: gZ^2/2, H H H: -3 mH^2/v).
template <class T, class C_>
HG_HD cx<T> vvsxxx(const Vc<T>& v1, const Vc<T>& v2, cx<T> s, C_ g) {
  return g * (s * vdot(v1, v2));
}
// jvsxxx: off-shell vector from a vector and a scalar
template <bool UNITARY, class T, class D, class R, class C_>
HG_HD Vc<T> jvsxxx(const Vc<T>& v, cx<T> s, C_ g, const Mom<T>& q, R rm2, D d) {
  const cx<T> gs = g * s;
  Vc<T> j;
  for (int i = 0; i < 4; ++i) j.c[i] = gs * v.c[i];
  return vprop<UNITARY>(j, q, rm2, d);
}
// hvvxxx: off-shell scalar from two vectors; d = -1/(q^2 - m^2 + i m Gamma)
template <class T, class D, class C_>
HG_HD cx<T> hvvxxx(const Vc<T>& v1, const Vc<T>& v2, C_ g, D d) {
  return d * (g * vdot(v1, v2));
}
template <class T>
HG_HD cx<T> vvssxx(const Vc<T>& v1, const Vc<T>& v2, cx<T> s3, cx<T> s4, T g) {
  return g * (s3 * s4 * vdot(v1, v2));
}
template <bool UNITARY, class T, class D, class R>
HG_HD Vc<T> jvssxx(const Vc<T>& v, cx<T> s3, cx<T> s4, T g, const Mom<T>& q, R rm2, D d) {
  return jvsxxx<UNITARY>(v, s3 * s4, g, q, rm2, d);
}
template <class T, class D>
HG_HD cx<T> hvvsxx(const Vc<T>& v1, const Vc<T>& v2, cx<T> s, T g, D d) {
  return d * (g * (s * vdot(v1, v2)));
}
template <class T, class C_>
HG_HD cx<T> sssxxx(cx<T> s1, cx<T> s2, cx<T> s3, C_ g) {
  return g * (s1 * s2 * s3);
}
template <class T, class D, class C_>
HG_HD cx<T> hssxxx(cx<T> s1, cx<T> s2, C_ g, D d) {
  return d * (g * (s1 * s2));
}

}  // namespace hg
