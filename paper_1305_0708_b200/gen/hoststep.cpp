// hoststep.cpp -- measurement tool: the GENERATED matrix elements and phase-space code compiled for the host
// (g++ -O3 -fopenmp) and run over the CPU cores, one pass of the hot path per call: Philox -> momenta -> cuts ->
// |Mbar|^2 -> weight -> (sum w, sum w^2, n_pass).  bench.py reports its events/s as `cpu_generated_code`: what a
// compiled CPU implementation of the SAME algorithm (shared sub-currents, non-zero helicities only, colour-flow
// basis) does on the box's cores -- the counterpart of the paper's Fortran HELAS baseline.
// It is not the oracle (bench.py's cpu_baseline) and not part of the product: never linked into libhg.so, no entry
// point of the library reaches it.
//   usage : hoststep <pid> <sqrt_s> <seed> <first_event> <n>
//   output: "<sum w> <sum w^2> <n_pass> <seconds> <threads>"
#include <omp.h>
#include <stdio.h>
#include <stdlib.h>

#include <chrono>
#include <vector>

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
int run(double rs, unsigned long long seed, unsigned long long first, long long n) {
  hg_params par;
  default_params(&par);
  hg_cuts cuts;
  default_cuts(P::pid, &cuts);
  const Coup<double> c = derive_couplings(par);
  const PsConst k = make_psconst(par, cuts, P::n_rambo, rs);
  const double wscale = kHbarC2Pb / (2.0 * rs * rs);
  double sw = 0.0, sw2 = 0.0, np = 0.0;
  const auto t0 = std::chrono::steady_clock::now();
#pragma omp parallel reduction(+ : sw, sw2, np)
  {
    std::vector<double> area(P::n_stage + 1);
    const HostStage<double> st{area.data()};
#pragma omp for schedule(static)
    for (long long e = 0; e < n; ++e) {
      Mom<double> p[P::n_ext];
      const double wps = P::gen(k, seed, first + (unsigned long long)e, p);
      if (!passes_cuts<P>(k, p)) continue;
      const double w = P::template me2<double>(p, c, st) * wps * wscale;
      sw += w;
      sw2 += w * w;
      np += 1.0;
    }
  }
  const double sec = std::chrono::duration<double>(std::chrono::steady_clock::now() - t0).count();
  printf("%.17g %.17g %.0f %.6f %d\n", sw, sw2, np, sec, omp_get_max_threads());
  return 0;
}

int main(int argc, char** argv) {
  if (argc != 6) {
    fprintf(stderr, "usage: hoststep <pid> <sqrt_s> <seed> <first_event> <n>\n");
    return 2;
  }
  const int pid = atoi(argv[1]);
  const double rs = atof(argv[2]);
  const unsigned long long seed = strtoull(argv[3], nullptr, 10), first = strtoull(argv[4], nullptr, 10);
  const long long n = atoll(argv[5]);
  switch (pid) {
    case 1: return run<P1>(rs, seed, first, n);
    case 2: return run<P2>(rs, seed, first, n);
    case 3: return run<P3>(rs, seed, first, n);
    case 4: return run<P4>(rs, seed, first, n);
    case 5: return run<P5>(rs, seed, first, n);
    case 6: return run<P6>(rs, seed, first, n);
    case 7: return run<P7>(rs, seed, first, n);
    case 8: return run<P8>(rs, seed, first, n);
    case 9: return run<P9>(rs, seed, first, n);
    case 10: return run<P10>(rs, seed, first, n);
    case 11: return run<P11>(rs, seed, first, n);
  }
  return 2;
}
