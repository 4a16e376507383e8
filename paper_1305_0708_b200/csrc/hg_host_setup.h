// hg_host_setup.h -- host-side preparation of per-call constants (shared by hg_api.cu and gen/flopcount.cpp).
#pragma once
#include <math.h>

#include "../../include/hg.h"
#include "hg_phase_space.cuh"

namespace hg {

constexpr double kHbarC2Pb = 0.3893793721e9;  // (hbar c)^2 in pb GeV^2

inline void default_params(hg_params* p) {
  p->mz = 91.1876;
  p->mw = 80.419;
  p->gz = 2.441;
  p->gw = 2.048;
  p->mt = 174.3;
  p->gt = 1.5;
  p->mb = 0.0;
  p->mh = 125.0;
  p->gh = 0.00407;
  p->alpha_em_inv = 132.507;
  p->alpha_s = 0.118;
  p->ckm_diagonal = 1;
  p->complex_mass = 0;
}

// BASELINE.json configs; scope readings SURVEY.md 8c-A11/A12.
inline bool default_cuts(int process, hg_cuts* c) {
  switch (process) {
    case HG_UDX_EPVE: *c = hg_cuts{0.0, 0.0, 0.0, 0.0}; return true;
    case HG_UUX_EPEMG: *c = hg_cuts{20.0, 2.5, 2.5, 0.0}; return true;
    case HG_UDX_EPVEGG: *c = hg_cuts{20.0, 0.0, 0.0, 0.4}; return true;
    case HG_GG_TTXG_DILEP: *c = hg_cuts{20.0, 2.5, 0.0, 0.0}; return true;
    case HG_UDX_EPVEGGG:
    case HG_UDX_EPVEGGGG: *c = hg_cuts{20.0, 2.5, 0.0, 0.4}; return true;
    case HG_UDX_EPVEH:
    case HG_UUX_EPEMHH:
    case HG_GG_TTXH:
    case HG_UD_HUD:
    case HG_UD_HHUD: *c = hg_cuts{0.0, 0.0, 0.0, 0.0}; return true;
  }
  return false;
}

inline bool default_hadronic(int process, hg_hadronic* h) {
  const double val[3] = {2.2, 0.5, 3.0}, sea[3] = {0.2, 1.2, 7.0}, glu[3] = {3.0, 1.2, 5.0};
  if (process < 1 || process > HG_N_PROCESS) return false;
  const double* a = process == HG_GG_TTXG_DILEP ? glu : val;
  const double* b = process == HG_GG_TTXG_DILEP ? glu : sea;
  h->y_res_max = 4.0;
  h->pdf_norm[0] = a[0];
  h->pdf_a[0] = a[1];
  h->pdf_b[0] = a[2];
  h->pdf_norm[1] = b[0];
  h->pdf_a[1] = b[1];
  h->pdf_b[1] = b[2];
  return true;
}

// n_rambo = number of momenta the RAMBO stage generates (n_final, or 3 for config 4).
inline PsConst make_psconst(const hg_params& par, const hg_cuts& cuts, int n_rambo, double rs) {
  PsConst k;
  k.rs = rs;
  k.vol = rambo_volume(n_rambo, rs);
  k.mt = par.mt;
  k.mgt = par.mt * par.gt;
  k.mw = par.mw;
  k.mgw = par.mw * par.gw;
  k.mb2 = par.mb * par.mb;
  k.mh = par.mh;
  k.tmax_t = par.gt > 0 ? atan(fmin(20.0, par.mt / par.gt)) : 0.0;
  k.tmax_w = par.gw > 0 ? atan(fmin(20.0, par.mw / par.gw)) : 0.0;
  k.pt_jet_min = cuts.pt_jet_min;
  k.eta_jet_max = cuts.eta_jet_max;
  k.eta_lep_max = cuts.eta_lep_max;
  k.dr_jj_min = cuts.dr_jj_min;
  k.grid = nullptr;
  k.nb = 0;
  k.had = 0;
  k.mz = par.mz;
  k.mgz = par.mz * par.gz;
  k.tmax_z = par.gz > 0 ? atan(fmin(20.0, par.mz / par.gz)) : 0.0;
  k.y_jet_max = cuts.eta_jet_max > 0 ? cuts.eta_jet_max : 5.0;
  const double ptmin = cuts.pt_jet_min > 0 ? cuts.pt_jet_min : 1.0;
  k.lnpt_lo = log(ptmin * ptmin);
  k.lnpt_hi = log(0.25 * rs * rs);
  k.y_res_max = 0.0;
  for (int i = 0; i < 2; ++i) {
    k.pdf_norm[i] = 1.0;
    k.pdf_a[i] = k.pdf_b[i] = 0.0;
  }
  return k;
}

}  // namespace hg
