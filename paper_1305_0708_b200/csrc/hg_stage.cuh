// hg_stage.cuh -- per-event staging area for values that live across a helicity loop.
//
// The generated matrix element of a large process (W + 3 jets: 63 sub-currents, 54 amplitudes) has more values
// alive across its helicity loops than fit in 255 registers; left to ptxas they become 3-5 KB of spill slots per
// thread, which at 256 threads per SM is far larger than L1 (profiles/r01_notes.md: 105 GB of DRAM traffic per
// launch from spills alone).  The generator therefore places every value that is produced outside a loop and
// consumed inside it in a slot of this area and reloads it at each use, so that inside a loop body only the
// operands of the current call are in registers.
//
// Device: the area is shared memory, laid out [slot][thread] so that a warp reads 32 consecutive words (no bank
// conflicts).  Loads are volatile: the compiler may neither merge them nor hoist them out of the loops, which would
// recreate the long live ranges.  Host (gen/flopcount, tests): a plain array per event.
#pragma once
#include "hg_cx.cuh"

namespace hg {

// no staging (small processes): every access is a compile error, the generator emits none
struct NoStage {};

#if defined(__CUDACC__)
// NAMED: the rendezvous is a named barrier of the warps that share the event (bar.sync id, threads of the pair /
// team) instead of a block-wide __syncthreads(): pairs and teams of one block no longer wait for each other.
// PAIRS (fp32 only): the words are laid out [slot / 2][event][slot % 2], so that two consecutive words of an event
// with an even first slot -- a complex number -- are ONE 8-byte access (get2 / put2).  The fp32 kernels are bound by
// instruction issue and 16 % of their instructions were 4-byte shared-memory loads.
template <class T, int STRIDE, bool NAMED = false, int TEAM_THREADS = 64, bool PAIRS = false>
struct SmemStage {
  T* b;      // shared memory + index of the event in the block
  int half;  // which half of the innermost helicity loop this warp evaluates (pair split, hg_process_impl.cuh)
  int group; // which group of closings of the innermost loop body (group split, P::n_split == 4; else 0)
  __device__ __forceinline__ int lo() const { return half; }
  __device__ __forceinline__ int hi() const { return half + 1; }
  // does this warp evaluate the part of a shared phase dealt to warp h of the pair / team? (emit.py _render_shared)
  __device__ __forceinline__ bool own(int h) const { return half + 2 * group == h; }
  // does this warp evaluate group g of the closings of the innermost loop body? (emit.py _partition)
  __device__ __forceinline__ bool grp(int g) const { return group == g; }
  __device__ __forceinline__ int at(int s) const { return PAIRS ? (s >> 1) * (2 * STRIDE) + (s & 1) : s * STRIDE; }
  __device__ __forceinline__ T get(int s) const { return ((volatile T*)b)[at(s)]; }
  __device__ __forceinline__ void put(int s, T v) const { b[at(s)] = v; }
  // words s and s + 1
  __device__ __forceinline__ void get2(int s, T& x, T& y) const {
    if constexpr (PAIRS) {
      static_assert(!PAIRS || sizeof(T) == 4, "paired layout: fp32 only");
      if ((s & 1) == 0) {   // s is a literal in the generated code: the test folds away
        const unsigned long long u = *(volatile const unsigned long long*)(b + at(s));
        x = __uint_as_float((unsigned)u);
        y = __uint_as_float((unsigned)(u >> 32));
        return;
      }
    }
    x = get(s);
    y = get(s + 1);
  }
  __device__ __forceinline__ void put2(int s, T x, T y) const {
    if constexpr (PAIRS) {
      if ((s & 1) == 0) {
        *(unsigned long long*)(b + at(s)) =
            (unsigned long long)__float_as_uint(x) | ((unsigned long long)__float_as_uint(y) << 32);
        return;
      }
    }
    put(s, x);
    put(s + 1, y);
  }
  // Block-wide rendezvous, emitted by the generator at the top of every helicity-loop iteration: the two warps of
  // a pair share the loop-level slots, so neither may start writing the values of the next iteration while the
  // other still reads those of the current one.  It also keeps the warps of a block close together in the code
  // (shared instruction-cache lines).  Every thread of the block must call me2().
  __device__ __forceinline__ void sync() const {
    if constexpr (NAMED) {
      const int id = 1 + (int)(threadIdx.x / TEAM_THREADS);   // barrier 0 is __syncthreads; at most 6 teams per block
      asm volatile("bar.sync %0, %1;" : : "r"(id), "n"(TEAM_THREADS) : "memory");
    } else {
      __syncthreads();
    }
  }
};
// Staging area in GLOBAL memory (P::stage_global: W + 4 jets, 738 words = 5.9 KB per event in fp64, which in shared
// memory leaves room for one pair of warps per SM).  Every block of the persistent grid owns a region laid out
// [slot][event of the block] like the shared-memory area, so a warp touches 32 consecutive words and slot s sits at
// the COMPILE-TIME offset s * STRIDE from one base pointer (with a run-time stride ptxas hoisted the 738 slot
// addresses out of the loops and spilled them: 13 KB of stack).  The accesses go to L2 (volatile: not cached in L1,
// not hoisted by the compiler); the working set of the grid, 592 blocks x 32 events x 5.9 KB = 112 MB, fits the
// 126 MB L2.  What is bought is occupancy: the number of warps is then limited by registers only.
template <class T, int STRIDE>
struct GmemStage {
  T* b;            // region of the block + event in the block
  int half;
  __device__ __forceinline__ int lo() const { return half; }
  __device__ __forceinline__ int hi() const { return half + 1; }
  __device__ __forceinline__ bool own(int h) const { return half == h; }
  __device__ __forceinline__ bool grp(int) const { return true; }   // pairs only: a warp runs every group in turn
  __device__ __forceinline__ T get(int s) const { return ((volatile T*)b)[s * STRIDE]; }
  __device__ __forceinline__ void put(int s, T v) const { ((volatile T*)b)[s * STRIDE] = v; }
  __device__ __forceinline__ void get2(int s, T& x, T& y) const { x = get(s); y = get(s + 1); }
  __device__ __forceinline__ void put2(int s, T x, T y) const { put(s, x); put(s + 1, y); }
  __device__ __forceinline__ void sync() const { __syncthreads(); }   // also orders the block's global accesses
};
#endif
template <class T>
struct HostStage {
  T* b;
  T get(int s) const { return b[s]; }
  void put(int s, T v) const { b[s] = v; }
  void get2(int s, T& x, T& y) const { x = b[s]; y = b[s + 1]; }
  void put2(int s, T x, T y) const { b[s] = x; b[s + 1] = y; }
  int lo() const { return 0; }
  int hi() const { return 2; }
  bool own(int) const { return true; }
  bool grp(int) const { return true; }
  void sync() const {}
};

template <class T, class St>
HG_HD T ld_T(const St& st, int s) {
  return st.get(s);
}
template <class T, class St>
HG_HD void st_T(const St& st, int s, T v) {
  st.put(s, v);
}
template <class T, class St>
HG_HD cx<T> ld_cx(const St& st, int s) {
  T re, im;
  st.get2(s, re, im);
  return mk<T>(re, im);
}
template <class T, class St>
HG_HD void st_cx(const St& st, int s, cx<T> v) {
  st.put2(s, v.re, v.im);
}
template <class T, class St>
HG_HD Mom<T> ld_mom(const St& st, int s) {
  T e, x, y, z;
  st.get2(s, e, x);
  st.get2(s + 2, y, z);
  return mkmom<T>(e, x, y, z);
}
template <class T, class St>
HG_HD void st_mom(const St& st, int s, const Mom<T>& v) {
  st.put2(s, v.e, v.x);
  st.put2(s + 2, v.y, v.z);
}
template <class T, class St>
HG_HD Vc<T> ld_vec(const St& st, int s) {
  Vc<T> v;
  for (int i = 0; i < 4; ++i) v.c[i] = ld_cx<T>(st, s + 2 * i);
  return v;
}
template <class T, class St>
HG_HD void st_vec(const St& st, int s, const Vc<T>& v) {
  for (int i = 0; i < 4; ++i) st_cx<T>(st, s + 2 * i, v.c[i]);
}
// spinor with slot mask M: only the non-zero slot pair(s) are kept
template <int M, class T, class St>
HG_HD Sp<T> ld_sp(const St& st, int s) {
  Sp<T> f;
  for (int i = 0; i < 4; ++i) f.c[i] = czero<T>();
  int o = s;
  if (M & SLOT_A) {
    f.c[0] = ld_cx<T>(st, o);
    f.c[1] = ld_cx<T>(st, o + 2);
    o += 4;
  }
  if (M & SLOT_B) {
    f.c[2] = ld_cx<T>(st, o);
    f.c[3] = ld_cx<T>(st, o + 2);
  }
  return f;
}
template <int M, class T, class St>
HG_HD void st_sp(const St& st, int s, const Sp<T>& f) {
  int o = s;
  if (M & SLOT_A) {
    st_cx<T>(st, o, f.c[0]);
    st_cx<T>(st, o + 2, f.c[1]);
    o += 4;
  }
  if (M & SLOT_B) {
    st_cx<T>(st, o, f.c[2]);
    st_cx<T>(st, o + 2, f.c[3]);
  }
}
// colour-flow accumulators kept in the staging area (processes with many flows): (X, Y) += k (rb, ib)
template <class T, class St>
HG_HD void acc_add(const St& st, int s, T k, cx<T> rb, cx<T> ib) {
  st.put(s, st.get(s) + k * rb.re);
  st.put(s + 1, st.get(s + 1) + k * rb.im);
  st.put(s + 2, st.get(s + 2) + k * ib.re);
  st.put(s + 3, st.get(s + 3) + k * ib.im);
}
// Op calls (gen/emit.py, option opcalls): the generated op functions of a process are REAL functions on the device
// (arguments and results by value: the ABI keeps them in registers), so that the innermost loop body is a sequence
// of short call sites instead of hundreds of KB of inlined arithmetic.
#if defined(__CUDACC__)
#define HG_OPCALL __host__ __device__ __noinline__
#else
#define HG_OPCALL inline
#endif
// what a closing returns: the projections on eps(+1) of the closing leg and on its conjugate (hg_helas.cuh close_proj)
template <class T>
struct RbIb {
  cx<T> rb, ib;
};
// the non-zero half of a single-chirality spinor (slot mask M = SLOT_A or SLOT_B): what an op function passes
template <class T>
struct Sh {
  cx<T> c[2];
};
template <int M, class T>
HG_HD Sh<T> sp_half(const Sp<T>& f) {
  constexpr int o = (M & SLOT_A) ? 0 : 2;
  Sh<T> h;
  h.c[0] = f.c[o];
  h.c[1] = f.c[o + 1];
  return h;
}
template <int M, class T>
HG_HD Sp<T> sp_full(const Sh<T>& h) {
  constexpr int o = (M & SLOT_A) ? 0 : 2;
  Sp<T> f;
  for (int i = 0; i < 4; ++i) f.c[i] = czero<T>();
  f.c[o] = h.c[0];
  f.c[o + 1] = h.c[1];
  return f;
}
// the same for N flows at once (offsets off[], factors k[]): all 4 N loads first, then the adds and stores, so that
// one shared-memory latency is paid per batch instead of one per flow
template <int N, class T, class St>
HG_HD void acc_add_batch(const St& st, int A, const int (&off)[N], const T (&k)[N], cx<T> rb, cx<T> ib) {
  T v[4 * N];
#pragma unroll
  for (int i = 0; i < N; ++i)
#pragma unroll
    for (int j = 0; j < 4; ++j) v[4 * i + j] = st.get(A + off[i] + j);
#pragma unroll
  for (int i = 0; i < N; ++i) {
    st.put(A + off[i], v[4 * i] + k[i] * rb.re);
    st.put(A + off[i] + 1, v[4 * i + 1] + k[i] * rb.im);
    st.put(A + off[i] + 2, v[4 * i + 2] + k[i] * ib.re);
    st.put(A + off[i] + 3, v[4 * i + 3] + k[i] * ib.im);
  }
}
// polarisation vector of a massless vector leg, helicity +1: eps^0 = 0 and eps^3 is real, so 5 words.
// flip != 0 returns the helicity -1 vector -conj(eps) (vflip).
template <class T, class St>
HG_HD void st_pol(const St& st, int s, const Vc<T>& e) {
  st.put2(s, e.c[1].re, e.c[1].im);
  st.put2(s + 2, e.c[2].re, e.c[2].im);
  st.put(s + 4, e.c[3].re);
}
template <class T, class St>
HG_HD Vc<T> ld_pol(const St& st, int s, int flip) {
  Vc<T> v;
  v.c[0] = czero<T>();
  v.c[1] = ld_cx<T>(st, s);
  v.c[2] = ld_cx<T>(st, s + 2);
  v.c[3] = mk<T>(st.get(s + 4), T(0));
  v.c[1].re = hflip(v.c[1].re, flip);
  v.c[2].re = hflip(v.c[2].re, flip);
  v.c[3].re = hflip(v.c[3].re, flip);
  return v;
}

// the same in the light-cone form the FFV vertices use (hg_helas.cuh Pol<T>; declared there, defined via the staged
// five words): flip != 0 gives the helicity -1 vector
template <class T>
struct Pol;
template <class T, class St>
HG_HD Pol<T> ld_pol_lc(const St& st, int s, int flip) {
  const cx<T> e1 = ld_cx<T>(st, s), e2 = ld_cx<T>(st, s + 2);
  const T v1r = hflip(e1.re, flip), v1i = e1.im, v2r = hflip(e2.re, flip), v2i = e2.im;
  Pol<T> p;
  p.v3 = hflip(st.get(s + 4), flip);
  p.ur = mk<T>(v1r + v2i, v1i - v2r);
  p.ll = mk<T>(v1r - v2i, v1i + v2r);
  return p;
}

}  // namespace hg
