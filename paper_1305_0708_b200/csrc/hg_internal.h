// hg_internal.h -- interface between the C-ABI layer (hg_api.cu) and the per-process translation units
// (generated/hg_proc_<pid>.cu, one per process so that they compile in parallel).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/hg.h"
#include "hg_params.cuh"
#include "hg_phase_space.cuh"

namespace hg {

// Grid of the fused integrate kernel: persistent, HG_INT_BLOCKS_PER_SM blocks of HG_INT_THREADS per SM.
constexpr int kIntThreads = 128;
constexpr int kMaxPartialBlocks = 148 * 16;

struct ProcVTable {
  hg_process_info_t info;
  // hg_matrix_element: p [n_ext][4][n] -> me2 [n]
  cudaError_t (*me)(int prec, int64_t n, const void* d_p, void* d_me2, const Coup<double>& c, cudaStream_t s);
  // hg_gen_phase_space
  cudaError_t (*ps)(int prec, int64_t n, const PsConst& k, uint64_t seed, uint64_t first, void* d_p,
                    void* d_wps, uint8_t* d_pass, cudaStream_t s);
  // hg_integrate_step: writes nblocks x (sum w, sum w^2, n_pass) partials; wscale = (hbar c)^2 / (2 s_hat)
  cudaError_t (*integrate)(int prec, int64_t n, const PsConst& k, uint64_t seed, uint64_t first,
                           const Coup<double>& c, double wscale, double* d_partials, int nblocks,
                           cudaStream_t s);
  // resident blocks per SM of the fused kernel for this precision (occupancy query)
  cudaError_t (*int_blocks_per_sm)(int prec, int* out);
};

extern const ProcVTable hg_proc_1, hg_proc_2, hg_proc_3, hg_proc_4, hg_proc_5;

}  // namespace hg
