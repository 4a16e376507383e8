// hg_process_impl.cuh -- the three kernels of one process, instantiated by generated/hg_proc_<pid>.cu.
//
// P is the generated process descriptor: n_ext, n_final, pid, jets/leptons for the cuts, gen() (phase space),
// me2<T>() (the fused helicity+colour summed matrix element emitted by gen/emit.py).
//
// Design: one phase-space point per thread, as in the paper, but
//   * a single fused kernel per process (the paper splits long amplitudes into several kernels with state in
//     global memory, PAPER.md:669 -- a CUDA 4.2 limit, not needed here);
//   * momenta in HBM are structure-of-arrays p[leg][mu][event]: a warp reads 32 consecutive values per
//     component (one or two full 128-byte lines), every wavefunction lives in registers;
//   * hg_integrate_step never touches HBM per event: Philox -> momenta -> cuts -> |M|^2 -> weight stay in
//     registers, the block reduces (sum w, sum w^2, n_pass) with warp shuffles and writes one partial.
#pragma once
#include "hg_internal.h"

namespace hg {

template <class P, class T>
__global__ void __launch_bounds__(P::me_threads) me_kernel(const T* __restrict__ p, T* __restrict__ me2,
                                                           int64_t n, const Coup<T> c) {
  const int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= n) return;
  Mom<T> q[P::n_ext];
#pragma unroll
  for (int l = 0; l < P::n_ext; ++l)
    q[l] = mkmom<T>(p[(l * 4 + 0) * n + e], p[(l * 4 + 1) * n + e], p[(l * 4 + 2) * n + e], p[(l * 4 + 3) * n + e]);
  me2[e] = P::template me2<T>(q, c);
}

template <class P, class T>
__global__ void __launch_bounds__(128) ps_kernel(const PsConst k, uint64_t seed, uint64_t first, int64_t n,
                                                 T* __restrict__ p, T* __restrict__ wps,
                                                 uint8_t* __restrict__ pass) {
  const int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= n) return;
  Mom<double> q[P::n_ext];
  const double w = P::gen(k, seed, first + (uint64_t)e, q);
#pragma unroll
  for (int l = 0; l < P::n_ext; ++l) {
    p[(l * 4 + 0) * n + e] = T(q[l].e);
    p[(l * 4 + 1) * n + e] = T(q[l].x);
    p[(l * 4 + 2) * n + e] = T(q[l].y);
    p[(l * 4 + 3) * n + e] = T(q[l].z);
  }
  wps[e] = T(w);
  if (pass) pass[e] = passes_cuts<P>(k, q) ? 1 : 0;
}

// Block reduction of three doubles: warp shuffle, then one value per warp through shared memory.
__device__ __forceinline__ void block_reduce3(double& a, double& b, double& c) {
  __shared__ double sh[3][32];
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

template <class P, class T>
__global__ void __launch_bounds__(kIntThreads) integrate_kernel(const PsConst k, uint64_t seed, uint64_t first,
                                                                int64_t n, const Coup<T> c, double wscale,
                                                                double* __restrict__ partials) {
  double sw = 0.0, sw2 = 0.0, np = 0.0;
  const int64_t stride = (int64_t)gridDim.x * blockDim.x;
  for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < n; e += stride) {
    Mom<double> q[P::n_ext];
    const double wps = P::gen(k, seed, first + (uint64_t)e, q);
    if (passes_cuts<P>(k, q)) {  // a failing point has a null weight and no second chance
      Mom<T> qt[P::n_ext];
#pragma unroll
      for (int l = 0; l < P::n_ext; ++l) qt[l] = mkmom<T>(T(q[l].e), T(q[l].x), T(q[l].y), T(q[l].z));
      const double w = (double)P::template me2<T>(qt, c) * wps * wscale;
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

template <class P>
struct Launch {
  static cudaError_t me(int prec, int64_t n, const void* d_p, void* d_me2, const Coup<double>& c, cudaStream_t s) {
    const unsigned grid = (unsigned)((n + P::me_threads - 1) / P::me_threads);
    if (prec == HG_F64)
      me_kernel<P, double><<<grid, P::me_threads, 0, s>>>((const double*)d_p, (double*)d_me2, n, c);
    else
      me_kernel<P, float><<<grid, P::me_threads, 0, s>>>((const float*)d_p, (float*)d_me2, n, coup_cast<float>(c));
    return cudaGetLastError();
  }
  static cudaError_t ps(int prec, int64_t n, const PsConst& k, uint64_t seed, uint64_t first, void* d_p,
                        void* d_wps, uint8_t* d_pass, cudaStream_t s) {
    const unsigned grid = (unsigned)((n + 127) / 128);
    if (prec == HG_F64)
      ps_kernel<P, double><<<grid, 128, 0, s>>>(k, seed, first, n, (double*)d_p, (double*)d_wps, d_pass);
    else
      ps_kernel<P, float><<<grid, 128, 0, s>>>(k, seed, first, n, (float*)d_p, (float*)d_wps, d_pass);
    return cudaGetLastError();
  }
  static cudaError_t integrate(int prec, int64_t n, const PsConst& k, uint64_t seed, uint64_t first,
                               const Coup<double>& c, double wscale, double* d_partials, int nblocks,
                               cudaStream_t s) {
    if (prec == HG_F64)
      integrate_kernel<P, double><<<nblocks, kIntThreads, 0, s>>>(k, seed, first, n, c, wscale, d_partials);
    else
      integrate_kernel<P, float><<<nblocks, kIntThreads, 0, s>>>(k, seed, first, n, coup_cast<float>(c), wscale,
                                                                d_partials);
    return cudaGetLastError();
  }
  static cudaError_t int_blocks_per_sm(int prec, int* out) {
    if (prec == HG_F64)
      return cudaOccupancyMaxActiveBlocksPerMultiprocessor(out, integrate_kernel<P, double>, kIntThreads, 0);
    return cudaOccupancyMaxActiveBlocksPerMultiprocessor(out, integrate_kernel<P, float>, kIntThreads, 0);
  }
};

template <class P>
constexpr ProcVTable make_vtable(double flops_me, double flops_ps) {
  return ProcVTable{hg_process_info_t{P::n_ext, P::n_final, P::n_hel_total, P::n_hel_nonzero, P::n_diagrams,
                                      P::n_amplitudes, P::n_flows, P::n_draws, P::avg_factor, flops_me, flops_ps},
                    &Launch<P>::me, &Launch<P>::ps, &Launch<P>::integrate, &Launch<P>::int_blocks_per_sm};
}

}  // namespace hg
