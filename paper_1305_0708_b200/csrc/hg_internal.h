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
// events per chunk of the two-kernel step of staged processes (the chunk buffer is 233 MB for W + 3 jets, fp64)
constexpr int64_t kIntChunk = (int64_t)1 << 20;
// events per chunk of the copy/compute pipeline of hg_matrix_element_host
constexpr int64_t kHostChunk = (int64_t)1 << 19;

// Accumulation of the adaptive-grid histograms after a chunk of the split step (hg_api.cu: hist_kernel): for the
// passing events listed by (idx, cnt, range, nblocks) adds w^2 into the bin of every draw.
struct GridAcc {
  int nb;               // bins per variable
  double* d_partial;    // [blocks][n_draws][nb] per-block histograms
  double* d_hist;       // [n_draws][nb], caller-owned, added to
  cudaError_t launch(const uint8_t* d_bins, const double* d_w, const int* d_idx, const int* d_cnt, int64_t m,
                     int64_t range, int nblocks, int n_draws, cudaStream_t s) const;
};

struct ProcVTable {
  hg_process_info_t info;
  // hg_matrix_element: p [n_ext][4][n] -> me2 [n]
  // d_gstage / gblocks: global staging buffer and grid of processes that stage in global memory (gstage below)
  // ebeam > 0: d_p holds the final-state legs only, the incoming momenta are ebeam (1, 0, 0, +-1)
  cudaError_t (*me)(int prec, int64_t n, const void* d_p, void* d_me2, const Coup<double>& c, void* d_gstage,
                    int gblocks, double ebeam, cudaStream_t s);
  // hg_gen_phase_space
  cudaError_t (*ps)(int prec, int64_t n, const PsConst& k, uint64_t seed, uint64_t first, void* d_p,
                    void* d_wps, uint8_t* d_pass, cudaStream_t s);
  // hg_integrate_step: writes nblocks x (sum w, sum w^2, n_pass) partials; wscale = (hbar c)^2 / (2 s_hat)
  // ev (or NULL): 3 events per chunk, recorded on s before the phase-space kernel, between the two kernels and
  // after the matrix-element kernel (hg_set_profiling); a fused process records ev[0] and ev[2] around its kernel.
  // Split-step processes (and every process when ga != NULL) run the step as separate kernels per chunk of `chunk`
  // events through the caller's scratch buffer (momenta, weight, pass flag, ...); the others ignore scratch and chunk.
  // ga (or NULL): adaptive-grid step, histograms accumulated after each chunk.
  cudaError_t (*integrate)(int prec, int64_t n, const PsConst& k, uint64_t seed, uint64_t first,
                           const Coup<double>& c, double wscale, double* d_partials, int nblocks,
                           void* d_scratch, int64_t chunk, cudaEvent_t* ev, const GridAcc* ga, void* d_gstage,
                           cudaStream_t s);
  // resident blocks per SM of the kernel that evaluates the matrix element in the step (occupancy query); split:
  // the split step is forced (adaptive-grid steps run every process as separate kernels)
  cudaError_t (*int_blocks_per_sm)(int prec, bool split, int* out);
  // bytes of the chunk buffer of the split step for `chunk` events; grid: with the histogram sections
  size_t (*scratch_bytes)(int prec, int64_t chunk, bool grid);
  bool (*split_step)();
  bool (*has_hadronic)();   // the paper's hadronic phase space is implemented for this process
  // global staging buffer (W + 4 jets): blocks of the persistent grid and bytes; 0 / 0 if staged in shared memory
  cudaError_t (*gstage)(int prec, int n_sm, int* blocks, size_t* bytes);
};

extern const ProcVTable hg_proc_1, hg_proc_2, hg_proc_3, hg_proc_4, hg_proc_5, hg_proc_6, hg_proc_7, hg_proc_8, hg_proc_9,
    hg_proc_10, hg_proc_11;

}  // namespace hg
