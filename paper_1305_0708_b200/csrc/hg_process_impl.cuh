// hg_process_impl.cuh -- the three kernels of one process, instantiated by generated/hg_proc_<pid>.cu.
//
// P is the generated process descriptor: n_ext, n_final, pid, jets/leptons for the cuts, gen() (phase space),
// me2<T>() (the fused helicity+colour summed matrix element emitted by gen/emit.py).
//
// Design: one phase-space point per thread, as in the paper -- or per
// pair of warps for the staged processes -- and
//   * one matrix-element kernel per process (the paper splits long amplitudes into several kernels with state in
//     global memory, PAPER.md:669 -- a CUDA 4.2 limit, not needed here);
//   * momenta in HBM are structure-of-arrays p[leg][mu][event]: a warp reads 32 consecutive values per
//     component (one or two full 128-byte lines), every wavefunction lives in registers or the staging area;
//   * hg_integrate_step is one fused kernel (integrate_kernel: nothing per event touches HBM) for the small
//     processes, and per chunk a phase-space kernel, an ordered compaction and me_acc_kernel for the others
//     (P::split_step); the block reduces (sum w, sum w^2, n_pass) with warp shuffles and writes one partial.
#pragma once
#include "hg_internal.h"
#include "hg_stage.cuh"

namespace hg {

// Threads per block of a kernel that evaluates me2<T>.
//
// A staged process (P::n_stage > 0) keeps P::n_stage words per EVENT in shared memory, which is what limits the
// events in flight on an SM (227 KB).  Each event is evaluated by a PAIR of warps (pair split): warps 2g and 2g+1
// of a block hold the same 32 events, share their staging area, and take one iteration each of the innermost
// helicity loop (SmemStage::lo/hi), which is ~85 % of the work; the phases outside it are dealt to the two warps
// by the generator (SmemStage::own), results meeting in the staging area at the next rendezvous.  Two warps per scheduler are what hides the instruction-fetch
// stall at every 128-byte line of the 170 KB straight-line code (profiles/r01_notes.md section 3).
constexpr int kSmemPerSM = 227 * 1024;
// P::n_split == 4 (group split, W + 4 jets): a TEAM of four warps per 32 events, warp t of the team = (half t & 1,
// group t >> 1): each half of the innermost loop is evaluated by two warps that share out its closings.
template <class P>
constexpr int kSplit = P::n_stage > 0 ? P::n_split : 1;
constexpr int kGlobalStageThreads = 256;   // global staging area: 4 pairs per block walk the code together
// words per event of the staging area: an even number with the paired fp32 layout (P::stage_pairs, hg_stage.cuh)
template <class P>
constexpr int stage_words() {
  return P::stage_pairs ? ((P::n_stage + 1) & ~1) : P::n_stage;
}
template <class P, class T>
constexpr int stage_threads(int want) {
  if (P::n_stage == 0) return want;
  if (P::stage_global) return kGlobalStageThreads;
  // 32-event groups that fit on an SM, leaving room for the kernels' static shared memory (3 KB; a team of four
  // has comb of me2_event, 3 x EPB words, and the scratch of block_reduce3, 384 bytes: at most 1152 bytes)
  const int groups = (kSmemPerSM - (P::n_split == 4 ? 1152 : 3072)) / (stage_words<P>() * (int)sizeof(T) * 32);
  if (P::n_split == 4) return 128 * (groups >= 3 ? 3 : (groups >= 2 ? 2 : 1));   // one to three teams = 4, 8, 12 warps
  // 2, 4 or 6 pairs = 4, 8 or 12 warps: a multiple of the 4 schedulers (6 and 10 warps measured slower than 4 and 8)
  const int g = groups >= 6 ? 6 : (groups >= 4 ? 4 : (groups >= 2 ? 2 : 1));
  return 64 * g;
}
template <class P, class T, int THREADS>
constexpr size_t stage_bytes() {
  return P::stage_global ? 0 : (size_t)stage_words<P>() * sizeof(T) * (THREADS / kSplit<P>);
}
// index of this thread's event within the block, and whether this thread owns the event's result
template <class P>
__device__ __forceinline__ int ev_local() {
  if constexpr (P::n_stage > 0) return ((threadIdx.x / (32 * kSplit<P>)) << 5) | (threadIdx.x & 31);
  return threadIdx.x;
}
template <class P>
__device__ __forceinline__ bool ev_owner() {
  if constexpr (P::n_stage > 0) return ((threadIdx.x >> 5) % kSplit<P>) == 0;
  return true;
}

// me2 of one event.  Staged: the staging area of the event is shared memory laid out [slot][event] (hg_stage.cuh);
// every thread of the block must call; the total is returned to the owner thread of the pair.
// gstage: global staging buffer, one region of n_stage x EPB words per block (P::stage_global), else unused.
template <class P, class T, int THREADS>
__device__ __forceinline__ T me2_event(const Mom<T>* q, const Coup<T>& c, T* gstage) {
  if constexpr (P::n_stage > 0) {
    constexpr int S = kSplit<P>;
    constexpr int EPB = THREADS / S;
    extern __shared__ __align__(16) unsigned char hg_stage_smem[];
    __shared__ T comb[S - 1][EPB];
    const int ev = ev_local<P>();
    const int wt = (threadIdx.x >> 5) % S;     // warp of the pair / team
    const int half = wt & 1, group = wt >> 1;
    T r;
    if constexpr (P::stage_global) {
      const GmemStage<T, EPB> st{gstage + (int64_t)blockIdx.x * (P::n_stage * EPB) + ev, half};
      r = P::template me2<T>(q, c, st);
    } else {
      // rendezvous per pair in fp64 only: in fp32 (12 warps per SM) the block-wide barrier, which also keeps the
      // warps on the same instruction-cache lines, measured 2-4 % faster; in fp64 (8-12 warps) 2-3 % slower
      constexpr bool PAIRS = P::stage_pairs && sizeof(T) == 4;   // fp32: complex numbers in one 8-byte access
      const SmemStage<T, EPB, P::named_barrier && sizeof(T) == 8, 32 * S, PAIRS> st{
          reinterpret_cast<T*>(hg_stage_smem) + (PAIRS ? 2 * ev : ev), half, group};
      r = P::template me2<T>(q, c, st);
    }
    if (wt) comb[wt - 1][ev] = r;
    __syncthreads();
    if (!wt) {
#pragma unroll
      for (int i = 0; i < S - 1; ++i) r += comb[i][ev];   // fixed order: deterministic
    }
    __syncthreads();  // comb and the staging area are free for the next event (pair-level barriers here: no gain)
    return r;
  } else {
    return P::template me2<T>(q, c, NoStage{});
  }
}

// Grid: one block per EPB events, or (P::stage_global) a persistent grid that strides over the batches, each block
// keeping its EPB columns of the global staging buffer.
template <class P, class T, int THREADS>
// ebeam > 0: p holds the FINAL-STATE legs only (leg l at row l - 2) and the incoming momenta are ebeam (1, 0, 0, +-1)
// (hg_matrix_element_host_cm: 64 bytes per event less over PCIe); ebeam <= 0: all n_ext legs.
__global__ void __launch_bounds__(THREADS) me_kernel(const T* __restrict__ p, T* __restrict__ me2, int64_t n,
                                                     const Coup<T> c, T* gstage, T ebeam) {
  constexpr int EPB = THREADS / kSplit<P>;
  const int l0 = ebeam > T(0) ? 2 : 0;     // grid-uniform
  // one batch per block; only a persistent grid (global staging) strides over several
  const int64_t stride = P::stage_global ? (int64_t)gridDim.x * EPB : n;
  for (int64_t base = (int64_t)blockIdx.x * EPB; base < n; base += stride) {   // block-uniform
    const int64_t e0 = base + ev_local<P>();
    const int64_t e = e0 < n ? e0 : n - 1;  // no early exit: a staged me2 holds block-wide rendezvous
    Mom<T> q[P::n_ext];
    q[0] = mkmom<T>(ebeam, T(0), T(0), ebeam);
    q[1] = mkmom<T>(ebeam, T(0), T(0), -ebeam);
#pragma unroll
    for (int l = 0; l < P::n_ext; ++l)
      if (l >= l0)
        q[l] = mkmom<T>(p[((l - l0) * 4 + 0) * n + e], p[((l - l0) * 4 + 1) * n + e], p[((l - l0) * 4 + 2) * n + e],
                        p[((l - l0) * 4 + 3) * n + e]);
    const T r = me2_event<P, T, THREADS>(q, c, gstage);
    if (e0 < n && ev_owner<P>()) me2[e0] = r;
  }
}

// BEAMS = true: all n_ext legs are written (hg_gen_phase_space).  BEAMS = false (chunk buffer of the split step): only
// the final-state legs, leg l at row l - 2; the two incoming momenta are sqrt(s_hat)/2 (1, 0, 0, +-1) for every
// event and me_acc_kernel rebuilds them from its arguments (64 of the 224 + 9 bytes per event of W + 3 jets less
// to write and read back).  bins (or NULL): [n_draws][n] grid bins of the draws (adaptive-grid steps).
// GRID: sampling through the adaptive grid k.grid (a separate instantiation: the flat kernel keeps its 72 registers).
// HAD: the paper's hadronic phase space; the incoming energies then differ from event to event and, with
// BEAMS = false, are written to beams [2][n] (doubles) for me_acc_kernel.  A point with a null weight (x >= 1) fails.
template <class P, class T, class W, bool BEAMS, bool GRID, bool HAD>
__global__ void __launch_bounds__(128) ps_kernel(const PsConst k, uint64_t seed, uint64_t first, int64_t n,
                                                 T* __restrict__ p, W* __restrict__ wps,
                                                 uint8_t* __restrict__ pass, uint8_t* __restrict__ bins,
                                                 double* __restrict__ beams) {
  const int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= n) return;
  Mom<double> q[P::n_ext];
  uint8_t b[GRID ? P::n_draws : 1];
  const double w = P::template gen<GRID, HAD>(k, seed, first + (uint64_t)e, q, GRID && bins ? b : nullptr);
  constexpr int L0 = BEAMS ? 0 : 2;
#pragma unroll
  for (int l = L0; l < P::n_ext; ++l) {
    p[((l - L0) * 4 + 0) * n + e] = T(q[l].e);
    p[((l - L0) * 4 + 1) * n + e] = T(q[l].x);
    p[((l - L0) * 4 + 2) * n + e] = T(q[l].y);
    p[((l - L0) * 4 + 3) * n + e] = T(q[l].z);
  }
  wps[e] = W(w);
  if (pass) pass[e] = (passes_cuts<P>(k, q) && (!HAD || w > 0.0)) ? 1 : 0;
  if constexpr (HAD && !BEAMS) {
    beams[e] = q[0].e;
    beams[n + e] = q[1].e;
  }
  if constexpr (GRID) {
    if (bins) {
#pragma unroll
      for (int d = 0; d < P::n_draws; ++d) bins[(int64_t)d * n + e] = b[d];
    }
  }
}

// Block reduction of three doubles: warp shuffle, then one value per warp through shared memory.
__device__ __forceinline__ void block_reduce3(double& a, double& b, double& c) {
  __shared__ double sh[3][16];   // up to 12 warps per block (stage_threads)
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    a += __shfl_down_sync(0xffffffffu, a, o);
    b += __shfl_down_sync(0xffffffffu, b, o);
    c += __shfl_down_sync(0xffffffffu, c, o);
  }
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
  if (lane == 0) {
    sh[0][w] = a;
    sh[1][w] = b;
    sh[2][w] = c;
  }
  __syncthreads();
  if (w == 0) {
    a = lane < nw ? sh[0][lane] : 0.0;
    b = lane < nw ? sh[1][lane] : 0.0;
    c = lane < nw ? sh[2][lane] : 0.0;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      a += __shfl_down_sync(0xffffffffu, a, o);
      b += __shfl_down_sync(0xffffffffu, b, o);
      c += __shfl_down_sync(0xffffffffu, c, o);
    }
  }
}

// me2_event of a staged process holds block-wide rendezvous, so it cannot sit under the divergent `if (passes_cuts)`
// below: staged processes always take the split step.
template <class P, class T, int THREADS>
__global__ void __launch_bounds__(THREADS) integrate_kernel(const PsConst k, uint64_t seed, uint64_t first,
                                                                int64_t n, const Coup<T> c, double wscale,
                                                                double* __restrict__ partials) {
  static_assert(P::n_stage == 0 || P::split_step, "a staged matrix element needs the split step");
  double sw = 0.0, sw2 = 0.0, np = 0.0;
  const int64_t stride = (int64_t)gridDim.x * blockDim.x;
  for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < n; e += stride) {
    Mom<double> q[P::n_ext];
    const double wps = P::gen(k, seed, first + (uint64_t)e, q);
    if (passes_cuts<P>(k, q)) {  // a failing point has a null weight and no second chance
      Mom<T> qt[P::n_ext];
#pragma unroll
      for (int l = 0; l < P::n_ext; ++l) qt[l] = mkmom<T>(T(q[l].e), T(q[l].x), T(q[l].y), T(q[l].z));
      const double w = (double)me2_event<P, T, THREADS>(qt, c, nullptr) * wps * wscale;
      sw += w;
      sw2 += w * w;
      np += 1.0;
    }
  }
  block_reduce3(sw, sw2, np);
  if (threadIdx.x == 0) {
    partials[3 * blockIdx.x + 0] = sw;
    partials[3 * blockIdx.x + 1] = sw2;
    partials[3 * blockIdx.x + 2] = np;
  }
}

// Ordered compaction of the events that pass the cuts: block b owns the events [b*range, (b+1)*range) of the
// chunk and writes their indices, in order, to idx[b*range ...]; cnt[b] = how many.  me_acc_kernel block b then
// evaluates exactly those, so that no lane idles on a failed event (10 % of W + 3 jets) and the order of the sums
// stays fixed (deterministic results).
static __global__ void __launch_bounds__(256) compact_kernel(const uint8_t* __restrict__ pass, int64_t n, int64_t range,
                                                      int* __restrict__ idx, int* __restrict__ cnt) {
  __shared__ int wsum[8];
  __shared__ int base;
  const int64_t lo = (int64_t)blockIdx.x * range;
  const int64_t hi = lo + range < n ? lo + range : n;
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  if (threadIdx.x == 0) base = 0;
  __syncthreads();
  for (int64_t t = lo; t < hi; t += 256) {
    const int64_t e = t + threadIdx.x;
    const bool ok = e < hi && pass[e] != 0;
    const unsigned m = __ballot_sync(0xffffffffu, ok);
    if (lane == 0) wsum[w] = __popc(m);
    __syncthreads();
    int off = base;
    for (int i = 0; i < w; ++i) off += wsum[i];
    if (ok) idx[lo + off + __popc(m & ((1u << lane) - 1u))] = (int)e;
    __syncthreads();
    if (threadIdx.x == 0) {
      int tot = 0;
      for (int i = 0; i < 8; ++i) tot += wsum[i];
      base += tot;
    }
    __syncthreads();
  }
  if (threadIdx.x == 0) cnt[blockIdx.x] = base;
}

// Second half of the step of a staged process: reads the points the ps_kernel wrote (momenta as T, weight as
// double, pass flag), evaluates |M|^2 and reduces (sum w, sum w^2, n_pass) per block.  The two halves are separate
// kernels because the phase-space code wants ~70 registers at full occupancy while the staged matrix element
// runs at 5-6 warps per SM; the round trip through HBM is 32 n_ext + 9 bytes per event against >= 2e4 flops.
// A block skips me2 only if none of its events passes (every thread must reach the rendezvous inside me2).
// p holds the final-state legs only (ps_kernel<.., BEAMS = false>); ebeam = sqrt(s_hat)/2, or beams [2][n] = the
// energies of the two incoming partons of every event (hadronic phase space).  wout (or NULL): receives
// the final weight w [pb] of every passing event at its index (adaptive-grid steps: input of hist_kernel).
template <class P, class T, int THREADS>
__global__ void __launch_bounds__(THREADS) me_acc_kernel(const T* __restrict__ p, const double* __restrict__ wps,
                                                         const int* __restrict__ idx, const int* __restrict__ cnt,
                                                         int64_t n, int64_t range, const Coup<T> c, double wscale,
                                                         double ebeam, const double* __restrict__ beams, int add,
                                                         double* __restrict__ partials, double* __restrict__ wout,
                                                         T* gstage) {
  constexpr int EPB = THREADS / kSplit<P>;
  double sw = 0.0, sw2 = 0.0, np = 0.0;
  const int m = cnt[blockIdx.x];                    // passing events of this block's range, block-uniform
  const int* __restrict__ my = idx + (int64_t)blockIdx.x * range;
  for (int base = 0; base < m; base += EPB) {
    const int j = base + ev_local<P>();
    const bool ok = j < m;
    const int64_t e = my[ok ? j : m - 1];           // tail lanes recompute the last event (rendezvous inside me2)
    Mom<T> q[P::n_ext];
    const double ea = beams ? beams[e] : ebeam, eb = beams ? beams[n + e] : ebeam;
    q[0] = mkmom<T>(T(ea), T(0), T(0), T(ea));
    q[1] = mkmom<T>(T(eb), T(0), T(0), T(-eb));
#pragma unroll
    for (int l = 2; l < P::n_ext; ++l)
      q[l] = mkmom<T>(p[((l - 2) * 4 + 0) * n + e], p[((l - 2) * 4 + 1) * n + e], p[((l - 2) * 4 + 2) * n + e],
                      p[((l - 2) * 4 + 3) * n + e]);
    const double w = (double)me2_event<P, T, THREADS>(q, c, gstage) * wps[e] * wscale;
    if (ok && ev_owner<P>()) {
      sw += w;
      sw2 += w * w;
      np += 1.0;
      if (wout) wout[e] = w;
    }
  }
  block_reduce3(sw, sw2, np);
  if (threadIdx.x == 0) {
    if (add) {
      sw += partials[3 * blockIdx.x + 0];
      sw2 += partials[3 * blockIdx.x + 1];
      np += partials[3 * blockIdx.x + 2];
    }
    partials[3 * blockIdx.x + 0] = sw;
    partials[3 * blockIdx.x + 1] = sw2;
    partials[3 * blockIdx.x + 2] = np;
  }
}

template <class P>
struct Launch {
  template <class T>
  static constexpr int me_thr() { return stage_threads<P, T>(P::me_threads); }
  template <class T>
  static constexpr int int_thr() { return stage_threads<P, T>(kIntThreads); }

  template <class K>
  static cudaError_t allow_smem(K kernel, size_t bytes) {
    if (bytes <= 48 * 1024) return cudaSuccess;
    return cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
  }
  // gblocks: blocks of the persistent grid, d_gstage: global staging buffer (P::stage_global only, gstage())
  template <class T>
  static cudaError_t me_t(int64_t n, const void* d_p, void* d_me2, const Coup<T>& c, void* d_gstage, int gblocks,
                          double ebeam, cudaStream_t s) {
    constexpr int TH = me_thr<T>();
    constexpr size_t smem = stage_bytes<P, T, TH>();
    cudaError_t err = allow_smem(me_kernel<P, T, TH>, smem);
    if (err != cudaSuccess) return err;
    constexpr int EPB = TH / kSplit<P>;
    unsigned grid = (unsigned)((n + EPB - 1) / EPB);
    if (P::stage_global && grid > (unsigned)gblocks) grid = (unsigned)gblocks;
    me_kernel<P, T, TH><<<grid, TH, smem, s>>>((const T*)d_p, (T*)d_me2, n, c, (T*)d_gstage, T(ebeam));
    return cudaGetLastError();
  }
  static cudaError_t me(int prec, int64_t n, const void* d_p, void* d_me2, const Coup<double>& c, void* d_gstage,
                        int gblocks, double ebeam, cudaStream_t s) {
    if (prec == HG_F64) return me_t<double>(n, d_p, d_me2, c, d_gstage, gblocks, ebeam, s);
    return me_t<float>(n, d_p, d_me2, coup_cast<float>(c), d_gstage, gblocks, ebeam, s);
  }
  // Global staging buffer: resident blocks per SM of the two kernels that evaluate me2 (the smaller one) and the
  // bytes of a buffer for n_sm * that many blocks; 0 blocks / 0 bytes for processes that stage in shared memory.
  template <class T>
  static cudaError_t gstage_t(int n_sm, int* blocks, size_t* bytes) {
    *blocks = 0;
    *bytes = 0;
    if constexpr (P::n_stage > 0 && P::stage_global) {
      constexpr int TH = me_thr<T>();
      int a = 0, b = 0;
      cudaError_t err = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&a, me_kernel<P, T, TH>, TH, 0);
      if (err == cudaSuccess) err = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&b, me_acc_kernel<P, T, TH>, TH, 0);
      if (err != cudaSuccess) return err;
      const int per_sm = a < b ? a : b;
      *blocks = n_sm * (per_sm < 1 ? 1 : per_sm);
      *bytes = (size_t)*blocks * (TH / kSplit<P>) * P::n_stage * sizeof(T);
    }
    return cudaSuccess;
  }
  static cudaError_t gstage(int prec, int n_sm, int* blocks, size_t* bytes) {
    return prec == HG_F64 ? gstage_t<double>(n_sm, blocks, bytes) : gstage_t<float>(n_sm, blocks, bytes);
  }
  // the four (grid, hadronic) variants of the phase-space kernel are separate instantiations
  template <class T, class W, bool BEAMS>
  static void ps_launch(unsigned grid, const PsConst& k, uint64_t seed, uint64_t first, int64_t n, T* d_p, W* d_w,
                        uint8_t* d_pass, uint8_t* d_bins, double* d_beams, cudaStream_t s) {
    const bool g = k.grid != nullptr, h = k.had != 0;
    if constexpr (P::has_hadronic) {
      if (g && h)
        ps_kernel<P, T, W, BEAMS, true, true><<<grid, 128, 0, s>>>(k, seed, first, n, d_p, d_w, d_pass, d_bins, d_beams);
      if (!g && h)
        ps_kernel<P, T, W, BEAMS, false, true><<<grid, 128, 0, s>>>(k, seed, first, n, d_p, d_w, d_pass, d_bins, d_beams);
    }
    if (g && !h)
      ps_kernel<P, T, W, BEAMS, true, false><<<grid, 128, 0, s>>>(k, seed, first, n, d_p, d_w, d_pass, d_bins, d_beams);
    if (!g && !h)
      ps_kernel<P, T, W, BEAMS, false, false><<<grid, 128, 0, s>>>(k, seed, first, n, d_p, d_w, d_pass, d_bins, d_beams);
  }
  static cudaError_t ps(int prec, int64_t n, const PsConst& k, uint64_t seed, uint64_t first, void* d_p,
                        void* d_wps, uint8_t* d_pass, cudaStream_t s) {
    const unsigned grid = (unsigned)((n + 127) / 128);
    if (prec == HG_F64)
      ps_launch<double, double, true>(grid, k, seed, first, n, (double*)d_p, (double*)d_wps, d_pass, nullptr, nullptr, s);
    else
      ps_launch<float, float, true>(grid, k, seed, first, n, (float*)d_p, (float*)d_wps, d_pass, nullptr, nullptr, s);
    return cudaGetLastError();
  }
  // Layout of the chunk buffer of the split step (context-owned, hg_api.cu): final-state momenta [n_ext - 2][4][chunk]
  // of T | weight double[chunk] | index list int[chunk] | per-block counts int[kMaxPartialBlocks] | pass flags
  // u8[chunk] | adaptive-grid steps only: final weights double[chunk], grid bins u8[n_draws][chunk].
  struct Scratch {   // byte offsets of the sections, each 256-byte aligned
    size_t p, w, idx, cnt, ok, beams, wout, bins, total;
  };
  static Scratch scratch_layout(size_t el, int64_t chunk, bool grid) {
    auto up = [](size_t x) { return (x + 255) / 256 * 256; };
    Scratch L;
    L.p = 0;
    L.w = up((size_t)chunk * (P::n_ext - 2) * 4 * el);
    L.idx = L.w + up((size_t)chunk * 8);
    L.cnt = L.idx + up((size_t)chunk * 4);
    L.ok = L.cnt + up(sizeof(int) * kMaxPartialBlocks);
    L.beams = L.ok + up((size_t)chunk);
    L.wout = L.beams + up((size_t)chunk * 16);
    L.bins = L.wout + (grid ? up((size_t)chunk * 8) : 0);
    L.total = L.bins + (grid ? up((size_t)chunk * P::n_draws) : 0);
    return L;
  }
  static size_t scratch_bytes(int prec, int64_t chunk, bool grid) {
    return scratch_layout(prec == HG_F64 ? 8 : 4, chunk, grid).total;
  }
  template <class T>
  static cudaError_t integrate_t(int64_t n, const PsConst& k, uint64_t seed, uint64_t first, const Coup<T>& c,
                                 double wscale, double* d_partials, int nblocks, void* d_scratch, int64_t chunk,
                                 cudaEvent_t* ev, const GridAcc* ga, void* d_gstage, cudaStream_t s) {
    constexpr int TH = int_thr<T>();
    constexpr size_t smem = stage_bytes<P, T, TH>();
    if constexpr (!P::split_step) {
      if (!k.grid && !k.had) {   // grid / hadronic sampling always take the split step (the fused kernel has neither)
        if (ev) cudaEventRecord(ev[0], s);
        integrate_kernel<P, T, TH><<<nblocks, TH, smem, s>>>(k, seed, first, n, c, wscale, d_partials);
        if (ev) cudaEventRecord(ev[2], s);
        return cudaGetLastError();
      }
    }
    cudaError_t err = allow_smem(me_acc_kernel<P, T, TH>, smem);
    if (err != cudaSuccess) return err;
    char* base = (char*)d_scratch;
    const Scratch L = scratch_layout(sizeof(T), chunk, ga != nullptr);
    T* d_p = (T*)(base + L.p);                                     // [n_ext - 2][4][m]
    double* d_w = (double*)(base + L.w);
    int* d_idx = (int*)(base + L.idx);
    int* d_cnt = (int*)(base + L.cnt);
    uint8_t* d_ok = (uint8_t*)(base + L.ok);
    double* d_beams = k.had ? (double*)(base + L.beams) : nullptr;
    double* d_wout = ga ? (double*)(base + L.wout) : nullptr;
    uint8_t* d_bins = ga ? (uint8_t*)(base + L.bins) : nullptr;
    for (int64_t off = 0; off < n; off += chunk) {
      const int64_t m = n - off < chunk ? n - off : chunk;
      const int64_t range = (m + nblocks - 1) / nblocks;
      cudaEvent_t* e3 = ev ? ev + 3 * (off / chunk) : nullptr;
      if (e3) cudaEventRecord(e3[0], s);
      ps_launch<T, double, false>((unsigned)((m + 127) / 128), k, seed, first + (uint64_t)off, m, d_p, d_w, d_ok,
                                  d_bins, d_beams, s);
      compact_kernel<<<nblocks, 256, 0, s>>>(d_ok, m, range, d_idx, d_cnt);
      if (e3) cudaEventRecord(e3[1], s);
      me_acc_kernel<P, T, TH><<<nblocks, TH, smem, s>>>(d_p, d_w, d_idx, d_cnt, m, range, c, wscale, 0.5 * k.rs,
                                                        d_beams, off > 0 ? 1 : 0, d_partials, d_wout, (T*)d_gstage);
      if (e3) cudaEventRecord(e3[2], s);
      if (ga) {
        err = ga->launch(d_bins, d_wout, d_idx, d_cnt, m, range, nblocks, P::n_draws, s);
        if (err != cudaSuccess) return err;
      }
    }
    return cudaGetLastError();
  }
  static cudaError_t integrate(int prec, int64_t n, const PsConst& k, uint64_t seed, uint64_t first,
                               const Coup<double>& c, double wscale, double* d_partials, int nblocks,
                               void* d_scratch, int64_t chunk, cudaEvent_t* ev, const GridAcc* ga, void* d_gstage,
                               cudaStream_t s) {
    if (prec == HG_F64)
      return integrate_t<double>(n, k, seed, first, c, wscale, d_partials, nblocks, d_scratch, chunk, ev, ga,
                                 d_gstage, s);
    return integrate_t<float>(n, k, seed, first, coup_cast<float>(c), wscale, d_partials, nblocks, d_scratch, chunk,
                              ev, ga, d_gstage, s);
  }
  template <class T>
  static cudaError_t int_blocks_t(int* out, bool split) {
    constexpr int TH = int_thr<T>();
    constexpr size_t smem = stage_bytes<P, T, TH>();
    if constexpr (!P::split_step) {
      if (!split) return cudaOccupancyMaxActiveBlocksPerMultiprocessor(out, integrate_kernel<P, T, TH>, TH, smem);
    }
    cudaError_t err = allow_smem(me_acc_kernel<P, T, TH>, smem);
    if (err != cudaSuccess) return err;
    return cudaOccupancyMaxActiveBlocksPerMultiprocessor(out, me_acc_kernel<P, T, TH>, TH, smem);
  }
  static cudaError_t int_blocks_per_sm(int prec, bool split, int* out) {
    return prec == HG_F64 ? int_blocks_t<double>(out, split) : int_blocks_t<float>(out, split);
  }
  static bool split_step() { return P::split_step; }
  static bool has_hadronic() { return P::has_hadronic; }
};

template <class P>
constexpr ProcVTable make_vtable(double flops_me, double flops_ps) {
  return ProcVTable{hg_process_info_t{P::n_ext, P::n_final, P::n_hel_total, P::n_hel_nonzero, P::n_diagrams,
                                      P::n_amplitudes, P::n_flows, P::n_draws, P::avg_factor, flops_me, flops_ps},
                    &Launch<P>::me, &Launch<P>::ps, &Launch<P>::integrate, &Launch<P>::int_blocks_per_sm,
                    &Launch<P>::scratch_bytes, &Launch<P>::split_step, &Launch<P>::has_hadronic, &Launch<P>::gstage};
}

}  // namespace hg
