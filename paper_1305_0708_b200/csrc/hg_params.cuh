// hg_params.cuh -- couplings and masses as seen by the generated device code.
//
// Values are derived on the host in hg_api.cu:hg_set_params from hg_params (include/hg.h) with the tree-level
// relations of SURVEY.md 8c-A5/A6 and passed to the kernels by value (they end up in the constant bank).
// FFV couplings are the (gL, gR) = (gc[0], gc[1]) of Eq. 35.  Member names are referenced by
// gen/model.py.
#pragma once

namespace hg {

template <class T>
struct Coup {
  // strong
  T gs, mgs, gs2;  // g_s, -g_s (qqg: gL = gR = -g_s, Eq. 36-38), g_s^2
  // electroweak FFV
  T gwf;                       // W-fermion:  -g_W/sqrt2 (left only)
  T gau, gad, gal;             // photon: -e Q
  T gzuL, gzuR, gzdL, gzdR, gzlL, gzlR, gznL;  // Z: -g_Z (T3 - Q sw2),  +g_Z Q sw2
  // gauge and Higgs self couplings (library vertices; Table 16, Eq. 39, 50-52)
  T gwwa, gwwz, gtth, gwwh, gzzh, gwwhh, gzzhh, ghhh;
  // imaginary parts of the couplings that contain m_W, m_Z (complex-mass option, Eq. 55-56 PAPER.md:1066-1073;
  // zero otherwise) and the flag itself (1 or 0): the q q / m_V^2 term then uses m_V^2 - i m_V Gamma_V
  T gtth_i, gwwh_i, gzzh_i, ghhh_i, cms;
  // masses and widths
  T mz, wz, mw, ww, mt, wt, mh, wh;
};

template <class T, class U>
inline Coup<T> coup_cast(const Coup<U>& s) {
  Coup<T> d;
  const U* sp = reinterpret_cast<const U*>(&s);
  T* dp = reinterpret_cast<T*>(&d);
  for (unsigned i = 0; i < sizeof(Coup<U>) / sizeof(U); ++i) dp[i] = T(sp[i]);
  return d;
}

}  // namespace hg
