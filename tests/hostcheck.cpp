// hostcheck.cpp -- test harness (tests/test_generated_host.py): evaluates the generated matrix elements in fp64 on the
// HOST (the device library compiles as plain C++) for momenta read from stdin, so that the emitted code can be
// checked without a GPU (tests/test_generated_host.py).  Never linked into libhg.so.
//   input : lines "pid  E px py pz  E px py pz ..." (n_ext momenta, leg order of include/hg.h); a NEGATIVE pid
//           evaluates process -pid with the complex-mass option (hg_params.complex_mass = 1)
//   output: one line per input line, |Mbar|^2 with 17 significant digits
//   `hostcheck team`: a staged process is evaluated the way the kernels do it (csrc/hg_process_impl.cuh me2_event):
//   by P::n_split THREADS that play the warps of a pair / team -- thread t = (half t & 1, group t >> 1) -- on one
//   shared staging area, st.sync() being a barrier of the threads; the partial results are added in warp order.
#include <stdio.h>
#include <string.h>

#include <condition_variable>
#include <mutex>
#include <thread>
#include <vector>

#include "../paper_1305_0708_b200/gen/flopcount.h"
#include "../paper_1305_0708_b200/csrc/hg_couplings.h"
#include "../paper_1305_0708_b200/csrc/hg_host_setup.h"
#include "../paper_1305_0708_b200/csrc/generated/hg_proc_1.cuh"
#include "../paper_1305_0708_b200/csrc/generated/hg_proc_2.cuh"
#include "../paper_1305_0708_b200/csrc/generated/hg_proc_3.cuh"
#include "../paper_1305_0708_b200/csrc/generated/hg_proc_4.cuh"
#include "../paper_1305_0708_b200/csrc/generated/hg_proc_5.cuh"
#include "../paper_1305_0708_b200/csrc/generated/hg_proc_6.cuh"
#include "../paper_1305_0708_b200/csrc/generated/hg_proc_7.cuh"
#include "../paper_1305_0708_b200/csrc/generated/hg_proc_8.cuh"
#include "../paper_1305_0708_b200/csrc/generated/hg_proc_9.cuh"
#include "../paper_1305_0708_b200/csrc/generated/hg_proc_10.cuh"
#include "../paper_1305_0708_b200/csrc/generated/hg_proc_11.cuh"

using namespace hg;

static bool g_team = false;

struct Barrier {   // reusable barrier of n threads (C++17)
  std::mutex m;
  std::condition_variable cv;
  int n, waiting = 0;
  long generation = 0;
  explicit Barrier(int n_) : n(n_) {}
  void wait() {
    std::unique_lock<std::mutex> lk(m);
    const long g = generation;
    if (++waiting == n) {
      waiting = 0;
      ++generation;
      cv.notify_all();
    } else {
      cv.wait(lk, [&] { return generation != g; });
    }
  }
};
// the staging area as one warp of a pair / team sees it (SmemStage of csrc/hg_stage.cuh on the host)
struct TeamStage {
  double* b;
  int half, group;
  Barrier* bar;
  double get(int s) const { return ((volatile double*)b)[s]; }
  void put(int s, double v) const { ((volatile double*)b)[s] = v; }
  void get2(int s, double& x, double& y) const { x = get(s); y = get(s + 1); }
  void put2(int s, double x, double y) const { put(s, x); put(s + 1, y); }
  int lo() const { return half; }
  int hi() const { return half + 1; }
  bool own(int h) const { return half + 2 * group == h; }
  bool grp(int g) const { return group == g; }
  void sync() const { bar->wait(); }
};

template <class P>
bool eval(const Coup<double>& c) {
  Mom<double> p[P::n_ext];
  for (int l = 0; l < P::n_ext; ++l)
    if (scanf("%lf %lf %lf %lf", &p[l].e, &p[l].x, &p[l].y, &p[l].z) != 4) return false;
  static double area[P::n_stage + 1];
  if (g_team && P::n_stage > 0) {
    constexpr int S = P::n_split;
    for (int i = 0; i <= P::n_stage; ++i) area[i] = 1e300;   // nothing may be read before it is written
    Barrier bar(S);
    double part[S];
    std::vector<std::thread> th;
    for (int t = 0; t < S; ++t)
      th.emplace_back([&, t] {
        const TeamStage st{area, t & 1, t >> 1, &bar};
        part[t] = P::template me2<double>(p, c, st);
      });
    for (auto& x : th) x.join();
    double r = part[0];
    for (int t = 1; t < S; ++t) r += part[t];
    printf("%.17g\n", r);
    return true;
  }
  const HostStage<double> st{area};
  printf("%.17g\n", P::template me2<double>(p, c, st));
  return true;
}

int main(int argc, char** argv) {
  g_team = argc > 1 && strcmp(argv[1], "team") == 0;
  hg_params par;
  default_params(&par);
  const Coup<double> c0 = derive_couplings(par);
  par.complex_mass = 1;
  const Coup<double> c1 = derive_couplings(par);
  int pid;
  while (scanf("%d", &pid) == 1) {
    bool ok = false;
    const Coup<double>& c = pid < 0 ? c1 : c0;
    if (pid < 0) pid = -pid;
    switch (pid) {
      case 1: ok = eval<P1>(c); break;
      case 2: ok = eval<P2>(c); break;
      case 3: ok = eval<P3>(c); break;
      case 4: ok = eval<P4>(c); break;
      case 5: ok = eval<P5>(c); break;
      case 6: ok = eval<P6>(c); break;
      case 7: ok = eval<P7>(c); break;
      case 8: ok = eval<P8>(c); break;
      case 9: ok = eval<P9>(c); break;
      case 10: ok = eval<P10>(c); break;
      case 11: ok = eval<P11>(c); break;
    }
    if (!ok) return 1;
  }
  return 0;
}
