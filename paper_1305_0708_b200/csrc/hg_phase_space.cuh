// hg_phase_space.cuh -- on-device phase-space generation, weights and cuts (steps a1-a4).
//
// The paper states the problem as: one phase-space point per thread from that thread's random numbers, no
// rejection loop ("each thread has one chance"), a point that violates a cut gets a null
// weight, heavy resonances are factorised, dPhi = dPhi_prod prod_k ds_k/2pi dPhi(R_k -> f_k)
// (Eq. 25-26), with the Breit-Wigner map s = m^2 + m Gamma tan(theta) (Eq. 27,
// PAPER.md:384-386; A.13-A.15).  BASELINE.json fixes sqrt(s_hat) and asks for flat RAMBO
// instead of the paper's (y, pT, phi) parameterisation (reading SURVEY.md 8c-A16; draw layout and the
// constraint-surface projection A16b in DESIGN.md).
//
// Everything here is fp64 regardless of the precision of the matrix element: the conformal RAMBO map is
// ill-conditioned for nearly collinear q_i, and the cut decisions must not depend on the ME precision
// (reading A17: the fp32 matrix element consumes fp64 momenta rounded to fp32).
#pragma once
#include "hg_philox.cuh"

namespace hg {

#define HG_TWO_PI 6.283185307179586476925286766559

// The fp64 transcendental functions of the phase space are CALLED, not inlined: one copy each of log, sincospi,
// asinh and atan2 instead of five or six.  The flat W + 3 jets phase-space kernel executed 4,660 instructions per
// event with 3.3 instruction-fetch stalls per issue (profiles/r02_notes.md): its straight-line code did not fit the
// instruction cache.
#if defined(__CUDACC__)
#define HG_CALL static __host__ __device__ __noinline__
#else
#define HG_CALL inline
#endif
HG_CALL double hlog(double x) { return log(x); }
HG_CALL double hasinh(double x) { return asinh(x); }
HG_CALL double hatan2(double y, double x) { return atan2(y, x); }

// sin, cos of 2 pi u.  On the device sincospi(2u): exact argument reduction, so no call to the Payne-Hanek slow path
// of sincos() is left in the fused kernels (a real CALL inside the W+3 jets fp64 kernel made ptxas fall back to an
// all-on-stack allocation, profiles/r01_notes.md).
struct SinCos {
  double s, c;
};
HG_CALL SinCos hsincos2pi_call(double u) {
  SinCos r;
#if defined(__CUDA_ARCH__)
  sincospi(2.0 * u, &r.s, &r.c);
#else
  r.s = sin(HG_TWO_PI * u);
  r.c = cos(HG_TWO_PI * u);
#endif
  return r;
}
HG_HD void hsincos2pi(double u, double& s, double& c) {
  const SinCos r = hsincos2pi_call(u);   // returned in registers: no stack traffic for the two results
  s = r.s;
  c = r.c;
}

// Constants of one hg_gen_phase_space / hg_integrate_step call, prepared on the host.
struct PsConst {
  double rs;       // sqrt(s_hat)
  double vol;      // massless RAMBO volume V_n (constant weight)
  double mt, mgt;  // top: mass, mass*width
  double mw, mgw;  // W
  double mb2;      // m_b^2
  double mh;       // Higgs mass (final-state mass of the Higgs-sector processes)
  double tmax_t, tmax_w;  // atan(min(20, m/Gamma))  (A.15; reading A14)
  double pt_jet_min, eta_jet_max, eta_lep_max, dr_jj_min;  // cuts, <= 0 disables
  // adaptive grid of the integration step (hg_set_grid, reading A22): device array [n_draws][nb + 1] of bin edges in
  // [0, 1], or NULL for flat sampling
  const double* grid;
  int nb;
  // the paper's hadronic phase space (hg_set_hadronic, reading A23; Eq. 24-28, App. A): rs is then the HADRONIC
  // sqrt(s); ranges of the integration variables and the toy parton densities f(x) = N x^-a (1 - x)^b of the beams
  int had;                 // 0: RAMBO at fixed s_hat; 1: hadronic
  double mz, mgz, tmax_z;
  double y_jet_max, lnpt_lo, lnpt_hi, y_res_max;
  double pdf_norm[2], pdf_a[2], pdf_b[2];
};

// Grid-optimised sampling (role of the BASES grid; VEGAS algorithm, reading A22):
// uniform y picks bin i = floor(y nb) of variable d and the point x = g[i] + (y nb - i)(g[i+1] - g[i]) in it; the
// Jacobian is nb (g[i+1] - g[i]).  u is mapped in place; returns the product of the Jacobians; bins (if not NULL)
// receives the bin of every variable.  x stays strictly below 1 (RAMBO takes log x).
template <int ND>
HG_HD double grid_map(const PsConst& k, double* u, uint8_t* bins) {
  double jac = 1.0;
  const int nb = k.nb;
#pragma unroll
  for (int d = 0; d < ND; ++d) {
    const double t = u[d] * (double)nb;
    int i = (int)t;
    if (i > nb - 1) i = nb - 1;
    const double* g = k.grid + (size_t)d * (nb + 1) + i;
    const double lo = g[0], w = g[1] - lo;
    const double x = lo + (t - (double)i) * w;
    u[d] = x < 0.99999999999999988898 ? x : 0.99999999999999988898;  // 1 - 2^-53
    jac *= (double)nb * w;
    if (bins) bins[d] = (uint8_t)i;
  }
  return jac;
}

// isotropic massless momentum of energy e
HG_HD Mom<double> iso(double uc, double uf, double e) {
  double c = 2.0 * uc - 1.0;
  double st = sqrt(1.0 - c * c);
  double sf, cf;
  hsincos2pi(uf, sf, cf);
  return mkmom<double>(e, e * st * cf, e * st * sf, e * c);
}

// Flat RAMBO for N massless momenta with total (rs, 0): u[4i..4i+3] = (cos theta, phi, energy, energy) of
// q_i; conformal map to the rest frame and scale; then the projection A16b.  The weight is the constant V_N.
template <int N>
HG_HD void rambo_massless(const double* u, double rs, Mom<double>* p) {
  Mom<double> Q = mkmom<double>(0, 0, 0, 0);
#pragma unroll
  for (int i = 0; i < N; ++i) {
    p[i] = iso(u[4 * i], u[4 * i + 1], -hlog(u[4 * i + 2] * u[4 * i + 3]));
    Q = Q + p[i];
  }
  const double rM = 1.0 / sqrt(mdot(Q, Q));
  const double bx = -Q.x * rM, by = -Q.y * rM, bz = -Q.z * rM;
  const double x = rs * rM, g = Q.e * rM, a = 1.0 / (1.0 + g);
  double sx = 0, sy = 0, sz = 0;
#pragma unroll
  for (int i = 0; i < N; ++i) {
    const Mom<double> q = p[i];
    const double bq = bx * q.x + by * q.y + bz * q.z;
    const double f = q.e + a * bq;
    if (i < N - 1) {
      p[i].x = x * (q.x + bx * f);
      p[i].y = x * (q.y + by * f);
      p[i].z = x * (q.z + bz * f);
      sx += p[i].x;
      sy += p[i].y;
      sz += p[i].z;
    } else {  // A16b: the last 3-momentum closes the sum
      p[i].x = -sx;
      p[i].y = -sy;
      p[i].z = -sz;
    }
  }
  double esum = 0;
#pragma unroll
  for (int i = 0; i < N; ++i) {
    p[i].e = sqrt(p[i].x * p[i].x + p[i].y * p[i].y + p[i].z * p[i].z);
    esum += p[i].e;
  }
  const double lam = rs / esum;
#pragma unroll
  for (int i = 0; i < N; ++i) {
    p[i].e *= lam;
    p[i].x *= lam;
    p[i].y *= lam;
    p[i].z *= lam;
  }
}

HG_HD double rambo_volume(int n, double rs) {
  // V_n = (pi/2)^(n-1) s^(n-2) / ((n-1)! (n-2)!) (2 pi)^(4-3n)
  double v = 1.0, f1 = 1.0, f2 = 1.0;
  for (int i = 0; i < n - 1; ++i) v *= 1.5707963267948966;
  for (int i = 0; i < 2 * n - 4; ++i) v *= rs;
  for (int i = 2; i <= n - 1; ++i) f1 *= i;
  for (int i = 2; i <= n - 2; ++i) f2 *= i;
  v /= f1 * f2;
  const int e = 3 * n - 4;
  for (int i = 0; i < e; ++i) v /= HG_TWO_PI;
  return v;
}

// Massive RAMBO: rescale the massless 3-momenta by xi with sum_i sqrt(m_i^2 + xi^2 E_i^2) = rs (Newton), and
// the weight factor (sum|k|/rs)^(2N-3) prod(|k|/E) rs / sum(|k|^2/E)   (reading A16).
template <int N>
HG_HD double rambo_massive(const double* u, const double* m2, double msum, double rs, Mom<double>* k) {
  rambo_massless<N>(u, rs, k);
  double xi = sqrt(1.0 - (msum / rs) * (msum / rs));
  // at most 12 Newton steps (the oracle always takes 12); quadratic convergence reaches the fixed point in 4-6, after
  // which a step changes xi by at most an ulp: stop once the energy sum is met to 4 ulp
#pragma unroll 1
  for (int it = 0; it < 12; ++it) {
    double f = -rs, df = 0;
#pragma unroll
    for (int i = 0; i < N; ++i) {
      const double e2 = k[i].e * k[i].e;
      const double en = sqrt(m2[i] + xi * xi * e2);
      f += en;
      df += xi * e2 / en;
    }
    xi -= f / df;
    if (fabs(f) <= 8.9e-16 * rs) break;
  }
  double ksum = 0, prod = 1, den = 0;
#pragma unroll
  for (int i = 0; i < N; ++i) {
    const double ka = xi * k[i].e;
    const double en = sqrt(m2[i] + ka * ka);
    k[i] = mkmom<double>(en, xi * k[i].x, xi * k[i].y, xi * k[i].z);
    ksum += ka;
    prod *= ka / en;
    den += ka * ka / en;
  }
  const double r = ksum / rs;
  double pw = r;
  for (int i = 1; i < 2 * N - 3; ++i) pw *= r;
  return pw * prod * rs / den;
}

// Eq. 27: s = m^2 + m Gamma tan(theta), theta uniform in +-tmax; returns ds/(2 pi) Jacobian.
HG_HD double bw_mass(double u, double m, double mg, double tmax, double& s) {
  const double th = -tmax + 2.0 * tmax * u;
  s = m * m + mg * tan(th);
  const double d = s - m * m;
  return (d * d + mg * mg) / mg * (2.0 * tmax) / HG_TWO_PI;
}

// pr in the rest frame of P (mass M) -> frame where it moves with P; energy from the mass shell (A16b).
HG_HD Mom<double> boost_from_rest(const Mom<double>& pr, const Mom<double>& P, double M, double msq) {
  const double e = (P.e * pr.e + P.x * pr.x + P.y * pr.y + P.z * pr.z) / M;
  const double fac = (e + pr.e) / (P.e + M);
  Mom<double> o;
  o.x = pr.x + fac * P.x;
  o.y = pr.y + fac * P.y;
  o.z = pr.z + fac * P.z;
  o.e = sqrt(o.x * o.x + o.y * o.y + o.z * o.z + msq);
  return o;
}

// Isotropic two-body decay P (mass^2 M2) -> (m1sq, m2sq); returns dPhi_2 = |p*| / (4 pi M)  (Eq. 26).
HG_HD double two_body(const Mom<double>& P, double M2, double m1sq, double m2sq, double uc, double uf,
                      Mom<double>& p1, Mom<double>& p2) {
  const double M = sqrt(M2);
  const double t = M2 - m1sq - m2sq;
  const double pst = sqrt(t * t - 4.0 * m1sq * m2sq) / (2.0 * M);
  Mom<double> d = iso(uc, uf, pst);
  const Mom<double> a = mkmom<double>(sqrt(pst * pst + m1sq), d.x, d.y, d.z);
  const Mom<double> b = mkmom<double>(sqrt(pst * pst + m2sq), -d.x, -d.y, -d.z);
  p1 = boost_from_rest(a, P, M, m1sq);
  p2 = boost_from_rest(b, P, M, m2sq);
  return pst / (2.0 * HG_TWO_PI * M);
}

// ---------------------------------------------------------------- per-process generators
// Writes p[0..n_ext) (leg order of include/hg.h) and returns the phase-space weight.
// GRID: the call samples through the adaptive grid k.grid (compile-time, so that the flat kernels carry none of it)
template <int NFINAL, bool GRID>
HG_HD double gen_massless(const PsConst& k, uint64_t seed, uint64_t event, uint32_t pid, Mom<double>* p,
                          uint8_t* bins) {
  double u[4 * NFINAL];
  draw_uniforms<4 * NFINAL>(seed, event, pid, u);
  double jac = 1.0;
  if constexpr (GRID) jac = grid_map<4 * NFINAL>(k, u, bins);
  const double h = 0.5 * k.rs;
  p[0] = mkmom<double>(h, 0.0, 0.0, h);
  p[1] = mkmom<double>(h, 0.0, 0.0, -h);
  rambo_massless<NFINAL>(u, k.rs, p + 2);
  return k.vol * jac;
}

// Final states with massive particles (Higgs-sector processes): massive RAMBO, masses m[i] of the final legs.
template <int NFINAL, bool GRID>
HG_HD double gen_massive(const PsConst& k, uint64_t seed, uint64_t event, uint32_t pid, const double (&m)[NFINAL],
                         Mom<double>* p, uint8_t* bins) {
  double u[4 * NFINAL];
  draw_uniforms<4 * NFINAL>(seed, event, pid, u);
  double jac = 1.0;
  if constexpr (GRID) jac = grid_map<4 * NFINAL>(k, u, bins);
  const double h = 0.5 * k.rs;
  p[0] = mkmom<double>(h, 0.0, 0.0, h);
  p[1] = mkmom<double>(h, 0.0, 0.0, -h);
  double m2[NFINAL], msum = 0.0;
#pragma unroll
  for (int i = 0; i < NFINAL; ++i) {
    m2[i] = m[i] * m[i];
    msum += m[i];
  }
  return k.vol * jac * rambo_massive<NFINAL>(u, m2, msum, k.rs, p + 2);
}

// config 4: g g -> (t -> b (W+ -> e+ ve)) (t~ -> b~ (W- -> mu- vm~)) g.  Draws: 0-3 s_t, s_t~, s_W+, s_W-;
// 4-15 RAMBO(t*, t~*, g); 16,17 t* decay angles; 18,19 W+*; 20,21 t~*; 22,23 W-*.
template <bool GRID>
HG_HD double gen_ttxg_dilep(const PsConst& k, uint64_t seed, uint64_t event, uint32_t pid, Mom<double>* p,
                            uint8_t* bins) {
  double u[24];
  draw_uniforms<24>(seed, event, pid, u);
  double jac = 1.0;
  if constexpr (GRID) jac = grid_map<24>(k, u, bins);
  const double h = 0.5 * k.rs;
  p[0] = mkmom<double>(h, 0.0, 0.0, h);
  p[1] = mkmom<double>(h, 0.0, 0.0, -h);
  double st, stb, swp, swm;
  double w = jac * bw_mass(u[0], k.mt, k.mgt, k.tmax_t, st);
  w *= bw_mass(u[1], k.mt, k.mgt, k.tmax_t, stb);
  w *= bw_mass(u[2], k.mw, k.mgw, k.tmax_w, swp);
  w *= bw_mass(u[3], k.mw, k.mgw, k.tmax_w, swm);
  const double m2[3] = {st, stb, 0.0};
  Mom<double> q[3];
  w *= k.vol * rambo_massive<3>(u + 4, m2, sqrt(st) + sqrt(stb), k.rs, q);
  Mom<double> wp, wm;
  w *= two_body(q[0], st, k.mb2, swp, u[16], u[17], p[2], wp);
  w *= two_body(wp, swp, 0.0, 0.0, u[18], u[19], p[3], p[4]);
  w *= two_body(q[1], stb, k.mb2, swm, u[20], u[21], p[5], wm);
  w *= two_body(wm, swm, 0.0, 0.0, u[22], u[23], p[6], p[7]);
  p[8] = q[2];
  return w;
}


// ---------------------------------------------------------------- the paper's hadronic phase space (reading A23)
// Eq. 24 / A.7 for n particles: y[i] (i < n), ln(pT^2 + m^2) and phi (i < n - 1) given;
// particle n - 1 takes the recoil (A.9a).  Writes the momenta, x_a, x_b (A.9b, c) and returns
// 1 / (2 s (4 pi)^(2n-3)) prod_{i<n-1} (pT_i^2 + m_i^2)  (Eq. 28 / A.11: dpT^2 = (pT^2 + m^2) d ln(pT^2 + m^2)).
template <int N>
HG_HD double generalised_ps(const double* y, const double* lnpt2m, const double* phi, const double* m2, double rs,
                            Mom<double>* k, double& xa, double& xb) {
  double w = 1.0 / (2.0 * rs * rs);
  if (N == 1) w *= 2.0 * HG_TWO_PI;   // (4 pi)^-(2N-3) with 2N - 3 = -1
#pragma unroll
  for (int i = 0; i < 2 * N - 3; ++i) w *= 1.0 / (2.0 * HG_TWO_PI);
  double px = 0.0, py = 0.0, sp = 0.0, sm = 0.0;
#pragma unroll
  for (int i = 0; i < N; ++i) {
    double kx, ky, mt2;
    if (i < N - 1) {
      mt2 = exp(lnpt2m[i]);
      const double pt = sqrt(fmax(mt2 - m2[i], 0.0));
      double sf, cf;
      hsincos2pi(phi[i], sf, cf);           // phi[i] holds the uniform: angle = 2 pi u
      kx = pt * cf;
      ky = pt * sf;
      px += kx;
      py += ky;
      w *= mt2;
    } else {
      kx = -px;
      ky = -py;
      mt2 = m2[i] + kx * kx + ky * ky;
    }
    const double mt = sqrt(mt2);
    k[i] = mkmom<double>(mt * cosh(y[i]), kx, ky, mt * sinh(y[i]));
    sp += k[i].e + k[i].z;
    sm += k[i].e - k[i].z;
  }
  xa = sp / rs;
  xb = sm / rs;
  return w;
}

HG_HD double toy_pdf(double x, double norm, double a, double b) { return norm * pow(x, -a) * pow(1.0 - x, b); }

// incoming legs from x_a, x_b; parton densities and s / s_hat; a point with x >= 1 gets a null weight (A.10)
HG_HD double had_finish(const PsConst& k, double w, double xa, double xb, Mom<double>* p) {
  const double ea = 0.5 * k.rs * xa, eb = 0.5 * k.rs * xb;
  p[0] = mkmom<double>(ea, 0.0, 0.0, ea);
  p[1] = mkmom<double>(eb, 0.0, 0.0, -eb);
  if (!(xa < 1.0 && xb < 1.0)) return 0.0;
  const double fa = toy_pdf(xa, k.pdf_norm[0], k.pdf_a[0], k.pdf_b[0]);
  const double fb = toy_pdf(xb, k.pdf_norm[1], k.pdf_a[1], k.pdf_b[1]);
  return w * fa * fb / (xa * xb);
}

// W/Z + NJ jets (configs 1, 2, 3, 5, 9): draws 0: s_R; 1+3j, 2+3j, 3+3j: y, ln pT^2, phi of jet j; 1+3NJ: y_R;
// 2+3NJ, 3+3NJ: decay angles of R -> l l'.  Legs: 2, 3 = the leptons, 4.. = the jets.
template <int NJ, int NDRAW, bool GRID>
HG_HD double gen_had_vjets(const PsConst& k, uint64_t seed, uint64_t event, uint32_t pid, double mres, double mgres,
                           double tmax, Mom<double>* p, uint8_t* bins) {
  double u[NDRAW];
  draw_uniforms<NDRAW>(seed, event, pid, u);
  double jac = 1.0;
  if constexpr (GRID) jac = grid_map<NDRAW>(k, u, bins);
  double sR;
  double w = jac * bw_mass(u[0], mres, mgres, tmax, sR);
  constexpr int N = NJ + 1;
  double y[N], lnpt[N], phi[N], m2[N];
#pragma unroll
  for (int j = 0; j < NJ; ++j) {
    y[j] = k.y_jet_max * (2.0 * u[1 + 3 * j] - 1.0);
    lnpt[j] = k.lnpt_lo + (k.lnpt_hi - k.lnpt_lo) * u[2 + 3 * j];
    phi[j] = u[3 + 3 * j];
    m2[j] = 0.0;
    w *= (2.0 * k.y_jet_max) * (k.lnpt_hi - k.lnpt_lo);
  }
  y[NJ] = k.y_res_max * (2.0 * u[1 + 3 * NJ] - 1.0);
  w *= 2.0 * k.y_res_max;
  m2[NJ] = sR;
  lnpt[NJ] = phi[NJ] = 0.0;
  Mom<double> q[N];
  double xa, xb;
  w *= generalised_ps<N>(y, lnpt, phi, m2, k.rs, q, xa, xb);
  w *= two_body(q[NJ], sR, 0.0, 0.0, u[2 + 3 * NJ], u[3 + 3 * NJ], p[2], p[3]);
#pragma unroll
  for (int j = 0; j < NJ; ++j) p[4 + j] = q[j];
  return had_finish(k, w, xa, xb, p);
}

// config 4: draws 0-3: s_t, s_t~, s_W+, s_W-; 4-6: gluon; 7-9: y, ln(pT^2 + s_t), phi of t*; 10: y of t~*; 11-18: decays.
template <bool GRID>
HG_HD double gen_had_ttxg_dilep(const PsConst& k, uint64_t seed, uint64_t event, uint32_t pid, Mom<double>* p,
                                uint8_t* bins) {
  double u[24];
  draw_uniforms<24>(seed, event, pid, u);
  double jac = 1.0;
  if constexpr (GRID) jac = grid_map<24>(k, u, bins);
  double st, stb, swp, swm;
  double w = jac * bw_mass(u[0], k.mt, k.mgt, k.tmax_t, st);
  w *= bw_mass(u[1], k.mt, k.mgt, k.tmax_t, stb);
  w *= bw_mass(u[2], k.mw, k.mgw, k.tmax_w, swp);
  w *= bw_mass(u[3], k.mw, k.mgw, k.tmax_w, swm);
  double y[3], lnpt[3], phi[3], m2[3];
  y[0] = k.y_jet_max * (2.0 * u[4] - 1.0);
  lnpt[0] = k.lnpt_lo + (k.lnpt_hi - k.lnpt_lo) * u[5];
  phi[0] = u[6];
  w *= (2.0 * k.y_jet_max) * (k.lnpt_hi - k.lnpt_lo);
  y[1] = k.y_res_max * (2.0 * u[7] - 1.0);
  const double lt0 = log(st), lt1 = log(st + 0.25 * k.rs * k.rs);   // Eq. 28 from pT = 0 to sqrt(s)/2
  lnpt[1] = lt0 + (lt1 - lt0) * u[8];
  phi[1] = u[9];
  y[2] = k.y_res_max * (2.0 * u[10] - 1.0);
  w *= (2.0 * k.y_res_max) * (lt1 - lt0) * (2.0 * k.y_res_max);
  m2[0] = 0.0;
  m2[1] = st;
  m2[2] = stb;
  lnpt[2] = phi[2] = 0.0;
  Mom<double> q[3];
  double xa, xb;
  w *= generalised_ps<3>(y, lnpt, phi, m2, k.rs, q, xa, xb);
  Mom<double> wp, wm;
  w *= two_body(q[1], st, k.mb2, swp, u[11], u[12], p[2], wp);
  w *= two_body(wp, swp, 0.0, 0.0, u[13], u[14], p[3], p[4]);
  w *= two_body(q[2], stb, k.mb2, swm, u[15], u[16], p[5], wm);
  w *= two_body(wm, swm, 0.0, 0.0, u[17], u[18], p[6], p[7]);
  p[8] = q[0];
  return had_finish(k, w, xa, xb, p);
}

// ---------------------------------------------------------------- cuts (Eq. 8-11)
HG_HD double pt_of(const Mom<double>& p) { return sqrt(p.x * p.x + p.y * p.y); }
HG_HD double eta_of(const Mom<double>& p) { return hasinh(p.z / pt_of(p)); }
HG_HD double delta_r(const Mom<double>& a, const Mom<double>& b) {  // Eq. 9b
  const double pi = 0.5 * HG_TWO_PI;
  double dphi = hatan2(a.y, a.x) - hatan2(b.y, b.x);
  if (dphi > pi) dphi -= HG_TWO_PI;
  if (dphi < -pi) dphi += HG_TWO_PI;
  const double deta = eta_of(a) - eta_of(b);
  return sqrt(deta * deta + dphi * dphi);
}

// P supplies n_jets / jets[] (gluon legs) and n_leps / leps[] (charged leptons) -- scope A11/A12.
template <class P>
HG_HD bool passes_cuts(const PsConst& k, const Mom<double>* p) {
  bool ok = true;
#pragma unroll
  for (int a = 0; a < P::n_jets; ++a) {
    const Mom<double>& j = p[P::jet(a)];
    if (k.pt_jet_min > 0) ok = ok && (pt_of(j) > k.pt_jet_min);
    if (k.eta_jet_max > 0) ok = ok && (fabs(eta_of(j)) < k.eta_jet_max);
  }
  if (k.eta_lep_max > 0) {
#pragma unroll
    for (int a = 0; a < P::n_leps; ++a) ok = ok && (fabs(eta_of(p[P::lep(a)])) < k.eta_lep_max);
  }
  if (k.dr_jj_min > 0) {
#pragma unroll
    for (int a = 0; a < P::n_jets; ++a)
#pragma unroll
      for (int b = a + 1; b < P::n_jets; ++b) ok = ok && (delta_r(p[P::jet(a)], p[P::jet(b)]) > k.dr_jj_min);
  }
  return ok;
}

}  // namespace hg
