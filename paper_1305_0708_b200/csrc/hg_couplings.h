// hg_couplings.h -- host-side derivation of the couplings from the SM inputs (hg_set_params).
//
// Tree-level relations, reading SURVEY.md 8c-A5/A6 (the paper's own inputs: PAPER.md:1075):
//   sw2 = 1 - mw^2/mz^2, e = sqrt(4 pi alpha), gW = e/sw, gZ = e/(sw cw), gs = sqrt(4 pi alpha_s);
//   L = psibar gamma^mu (gL PL + gR PR) psi V_mu (Eq. 35) with
//   D_mu = d_mu + i e Q A_mu + i gZ (T3 - Q sw2) Z_mu + i gW/sqrt2 (W+ T+ + W- T-) + i gs T^a G^a_mu.
#pragma once
#include <math.h>

#include "../../include/hg.h"
#include "hg_params.cuh"

namespace hg {

inline Coup<double> derive_couplings(const hg_params& par) {
  const double pi = 3.14159265358979323846;
  Coup<double> c;
  double sw2 = 1.0 - (par.mw * par.mw) / (par.mz * par.mz);
  double sw = sqrt(sw2), cw = sqrt(1.0 - sw2);
  double e = sqrt(4.0 * pi / par.alpha_em_inv);
  double gw = e / sw, gz = e / (sw * cw);
  c.gs = sqrt(4.0 * pi * par.alpha_s);
  c.mgs = -c.gs;
  c.gs2 = c.gs * c.gs;
  c.gwf = -gw / sqrt(2.0);
  const double qu = 2.0 / 3.0, qd = -1.0 / 3.0, ql = -1.0;
  c.gau = -e * qu;
  c.gad = -e * qd;
  c.gal = -e * ql;
  c.gzuL = -gz * (0.5 - qu * sw2);
  c.gzuR = gz * qu * sw2;
  c.gzdL = -gz * (-0.5 - qd * sw2);
  c.gzdR = gz * qd * sw2;
  c.gzlL = -gz * (-0.5 - ql * sw2);
  c.gzlR = gz * ql * sw2;
  c.gznL = -gz * 0.5;
  // gauge self couplings (Table 16): gWWA = e, gWWZ = gW cw
  c.gwwa = e;
  c.gwwz = gw * cw;
  // Higgs couplings (Eq. 39, 50-52): v = 2 mw / gW.  Complex-mass option (Eq. 55-56; DESIGN.md
  // A4b): m_V -> mu_V = sqrt(m_V^2 - i m_V Gamma_V) in these couplings, with mu_W^2 = (gW^2/gZ^2) mu_Z^2 imposed:
  // gW^2/gZ^2 = cw^2 = mw^2/mz^2 is real here, so Eq. 56 fixes Gamma_W = mw Gamma_Z / mz (the input gw is ignored).
  const bool cms = par.complex_mass != 0;
  const double ww = cms ? par.mw * par.gz / par.mz : par.gw;
  // principal square root of m^2 - i m Gamma
  auto csqrt_ = [](double re, double im, double& ore, double& oim) {
    const double r = sqrt(re * re + im * im);
    ore = sqrt(0.5 * (r + re));
    oim = (im < 0 ? -1.0 : 1.0) * sqrt(0.5 * (r - re));
  };
  double mwr = par.mw, mwi = 0.0, mzr = par.mz, mzi = 0.0;
  if (cms) {
    csqrt_(par.mw * par.mw, -par.mw * ww, mwr, mwi);
    csqrt_(par.mz * par.mz, -par.mz * par.gz, mzr, mzi);
  }
  // 1 / v = gW / (2 mu_W)
  const double mw2abs = mwr * mwr + mwi * mwi;
  const double ivr = 0.5 * gw * mwr / mw2abs, ivi = -0.5 * gw * mwi / mw2abs;
  c.gtth = -par.mt * ivr;
  c.gtth_i = -par.mt * ivi;
  c.gwwh = gw * mwr;
  c.gwwh_i = gw * mwi;
  c.gzzh = gz * mzr;
  c.gzzh_i = gz * mzi;
  c.gwwhh = 0.5 * gw * gw;
  c.gzzhh = 0.5 * gz * gz;
  c.ghhh = -3.0 * par.mh * par.mh * ivr;
  c.ghhh_i = -3.0 * par.mh * par.mh * ivi;
  c.cms = cms ? 1.0 : 0.0;
  c.mz = par.mz;
  c.wz = par.gz;
  c.mw = par.mw;
  c.ww = ww;
  c.mt = par.mt;
  c.wt = par.gt;
  c.mh = par.mh;
  c.wh = par.gh;
  return c;
}

}  // namespace hg
