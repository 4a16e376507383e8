// flopcount.cpp -- build-time tool of the generator: runs every generated matrix element on the counting type
// (flopcount.h) over a few phase-space points produced by the library's own generator compiled for the host,
// and prints one line "pid flops_min flops_mean flops_max me2_double me2_counted" per process.
// Compiled and run by gen/processes.py:count_flops (g++), never linked into libhg.so.
#include <stdio.h>

#include "flopcount.h"
#include "../csrc/hg_couplings.h"
#include "../csrc/hg_host_setup.h"
#include "../csrc/generated/hg_proc_1.cuh"
#include "../csrc/generated/hg_proc_2.cuh"
#include "../csrc/generated/hg_proc_3.cuh"
#include "../csrc/generated/hg_proc_4.cuh"
#include "../csrc/generated/hg_proc_5.cuh"
#include "../csrc/generated/hg_proc_6.cuh"
#include "../csrc/generated/hg_proc_7.cuh"
#include "../csrc/generated/hg_proc_8.cuh"
#include "../csrc/generated/hg_proc_9.cuh"
#include "../csrc/generated/hg_proc_10.cuh"
#include "../csrc/generated/hg_proc_11.cuh"

using namespace hg;

template <class P>
void run(double rs) {
  hg_params par;
  default_params(&par);
  hg_cuts cuts;
  default_cuts(P::pid, &cuts);
  const Coup<double> cd = derive_couplings(par);
  const Coup<Cnt> cc = coup_cast<Cnt>(cd);
  const PsConst k = make_psconst(par, cuts, P::n_rambo, rs);
  long long lo = 0, hi = 0, sum = 0;
  double v_d = 0, v_c = 0;
  const int N = 32;
  for (int e = 0; e < N; ++e) {
    Mom<double> p[P::n_ext];
    P::gen(k, 20130507ull, (unsigned long long)e, p);
    Mom<Cnt> q[P::n_ext];
    for (int l = 0; l < P::n_ext; ++l) q[l] = mkmom<Cnt>(Cnt(p[l].e), Cnt(p[l].x), Cnt(p[l].y), Cnt(p[l].z));
    static Cnt sc[P::n_stage + 1];
    static double sd[P::n_stage + 1];
    const HostStage<Cnt> stc{sc};
    const HostStage<double> std_{sd};
    Cnt::n() = 0;
    const Cnt r = P::template me2<Cnt>(q, cc, stc);
    const long long f = Cnt::n();
    if (e == 0 || f < lo) lo = f;
    if (e == 0 || f > hi) hi = f;
    sum += f;
    v_c = r.v;
    v_d = P::template me2<double>(p, cd, std_);
  }
  printf("%d %lld %.1f %lld %.17g %.17g\n", P::pid, lo, (double)sum / N, hi, v_d, v_c);
}

int main() {
  run<P1>(80.0);
  run<P2>(500.0);
  run<P3>(1000.0);
  run<P4>(1500.0);
  run<P5>(2000.0);
  run<P6>(500.0);
  run<P7>(1000.0);
  run<P8>(1000.0);
  run<P9>(3000.0);
  run<P10>(1000.0);
  run<P11>(1000.0);
  return 0;
}
