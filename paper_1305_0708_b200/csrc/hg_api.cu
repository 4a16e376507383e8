// hg_api.cu -- the C-ABI boundary of libhg.so (include/hg.h): argument checking, per-call constants, dispatch to
// the per-process translation units, the process-independent kernels (accumulate, finalize, FMA peak).
#include <math.h>
#include <stdio.h>
#include <string.h>

#include <mutex>
#include <string>
#include <vector>

#include "../../include/hg_bench.h"
#include "hg_couplings.h"
#include "hg_host_setup.h"
#include "hg_internal.h"

namespace hg {

static const ProcVTable* vtable(int process) {
  switch (process) {
    case HG_UDX_EPVE: return &hg_proc_1;
    case HG_UUX_EPEMG: return &hg_proc_2;
    case HG_UDX_EPVEGG: return &hg_proc_3;
    case HG_GG_TTXG_DILEP: return &hg_proc_4;
    case HG_UDX_EPVEGGG: return &hg_proc_5;
    case HG_UDX_EPVEH: return &hg_proc_6;
    case HG_UUX_EPEMHH: return &hg_proc_7;
    case HG_GG_TTXH: return &hg_proc_8;
    case HG_UDX_EPVEGGGG: return &hg_proc_9;
    case HG_UD_HUD: return &hg_proc_10;
    case HG_UD_HHUD: return &hg_proc_11;
  }
  return nullptr;
}

static std::string g_create_error;

}  // namespace hg

struct hg_ctx {
  int device = 0;
  int n_sm = 0;
  bool params_set = false;
  hg_params par;
  hg_cuts cuts[HG_N_PROCESS + 1];
  bool cuts_user = false;
  hg::Coup<double> coup;
  double* d_partials = nullptr;  // [kMaxPartialBlocks][3]
  double* d_acc = nullptr;       // [3]
  double* h_acc = nullptr;       // pinned [3]
  void* d_stage = nullptr;       // staging for hg_matrix_element_host
  size_t stage_bytes = 0;
  void* d_scratch = nullptr;     // phase-space points of one chunk of hg_integrate_step (staged processes)
  size_t scratch_bytes = 0;
  bool hadronic = false;           // hg_set_hadronic
  hg_hadronic had;
  const double* d_grid = nullptr;  // hg_set_grid: caller-owned [grid_ndim][grid_nb + 1]
  int grid_nb = 0;
  int grid_ndim = 0;
  double* d_hist = nullptr;        // caller-owned [n_draws][grid_nb], or NULL
  void* d_gstage = nullptr;          // global staging buffer of processes that stage in global memory (W + 4 jets)
  size_t gstage_bytes = 0;
  double* d_hist_partial = nullptr;  // per-block histograms of one chunk
  size_t hist_partial_bytes = 0;
  cudaStream_t copy_stream = nullptr;   // H2D copies of hg_matrix_element_host
  cudaEvent_t ev_h2d[2] = {nullptr, nullptr}, ev_free[2] = {nullptr, nullptr};
  int profiling = 0;             // hg_set_profiling
  std::vector<cudaEvent_t> ev;   // 3 per chunk
  double t_ps_ms = 0, t_me_ms = 0;
  int n_launches = 0;            // kernels launched by the last hg_integrate_step
  std::string err;
};

namespace hg {

static int fail(hg_ctx* ctx, int code, const char* msg) {
  if (ctx) ctx->err = msg;
  return code;
}
static int fail_cuda(hg_ctx* ctx, cudaError_t e, const char* where) {
  if (ctx) ctx->err = std::string(where) + ": " + cudaGetErrorString(e);
  return HG_ECUDA;
}

// failures of calls that have no context: the text goes where hg_last_error(NULL) reads it
static int fail_noctx(int code, const char* msg) {
  g_create_error = msg;
  return code;
}
static int fail_cuda_noctx(cudaError_t e, const char* where) {
  g_create_error = std::string(where) + ": " + cudaGetErrorString(e);
  return HG_ECUDA;
}
constexpr int kNoAllocMaxDevices = 64;

// Sums nb x 3 partials in a fixed order (deterministic result for a given grid).
__global__ void finalize_kernel(const double* __restrict__ partials, int nb, double* __restrict__ acc) {
  __shared__ double sh[3][256];
  double a = 0, b = 0, c = 0;
  for (int i = threadIdx.x; i < nb; i += blockDim.x) {
    a += partials[3 * i];
    b += partials[3 * i + 1];
    c += partials[3 * i + 2];
  }
  sh[0][threadIdx.x] = a;
  sh[1][threadIdx.x] = b;
  sh[2][threadIdx.x] = c;
  __syncthreads();
  for (int s = blockDim.x / 2; s > 0; s >>= 1) {
    if ((int)threadIdx.x < s) {
      sh[0][threadIdx.x] += sh[0][threadIdx.x + s];
      sh[1][threadIdx.x] += sh[1][threadIdx.x + s];
      sh[2][threadIdx.x] += sh[2][threadIdx.x + s];
    }
    __syncthreads();
  }
  if (threadIdx.x == 0) {
    acc[0] = sh[0][0];
    acc[1] = sh[1][0];
    acc[2] = sh[2][0];
  }
}

// Steps a9-a10 on arrays: w = pass * me2 * wps * wscale.
template <class T>
__global__ void __launch_bounds__(256) accumulate_kernel(const T* __restrict__ me2, const T* __restrict__ wps,
                                                         const uint8_t* __restrict__ pass, int64_t n,
                                                         double wscale, double* __restrict__ partials) {
  __shared__ double sh[3][8];
  double sw = 0, sw2 = 0, np = 0;
  const int64_t stride = (int64_t)gridDim.x * blockDim.x;
  for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < n; e += stride) {
    const bool ok = pass ? pass[e] != 0 : true;
    if (ok) {
      const double w = (double)me2[e] * (double)wps[e] * wscale;
      sw += w;
      sw2 += w * w;
      np += 1.0;
    }
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    sw += __shfl_down_sync(0xffffffffu, sw, o);
    sw2 += __shfl_down_sync(0xffffffffu, sw2, o);
    np += __shfl_down_sync(0xffffffffu, np, o);
  }
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  if (lane == 0) {
    sh[0][w] = sw;
    sh[1][w] = sw2;
    sh[2][w] = np;
  }
  __syncthreads();
  if (threadIdx.x == 0) {
    double a = 0, b = 0, c = 0;
    for (int i = 0; i < 8; ++i) {
      a += sh[0][i];
      b += sh[1][i];
      c += sh[2][i];
    }
    partials[3 * blockIdx.x] = a;
    partials[3 * blockIdx.x + 1] = b;
    partials[3 * blockIdx.x + 2] = c;
  }
}

// ---- hg_accumulate_noalloc: steps a9-a10 with the partial sums in a file-scope device array (no allocation) ----
constexpr int kNoAllocRange = 4096;                                   // events per block (16 per thread)
constexpr int kNoAllocMaxBlocks = HG_NOALLOC_MAX_EVENTS / kNoAllocRange;   // 4096 blocks
// The scratch of hg_accumulate_noalloc: [kNoAllocMaxBlocks][3] partial sums, 96 KB per GPU that loads the library.
// In HOST code this name is a host-side stand-in, not a device address: the host passes the address it gets from
// cudaGetSymbolAddress (noalloc_scratch below), once per device.
static __device__ __align__(256) double hg_noalloc_partials[3 * kNoAllocMaxBlocks];

// accumulate_kernel with a fixed range of events per block (the grid, and so the order of the sums, does not
// depend on the number of SMs).  Every block writes its three entries, also when none of its events passes.
template <class T>
__global__ void __launch_bounds__(256) accumulate_noalloc_kernel(const T* __restrict__ me2, const T* __restrict__ wps,
                                                                 const uint8_t* __restrict__ pass, int64_t n,
                                                                 double wscale, double* __restrict__ partials) {
  __shared__ double sh[3][8];
  double sw = 0, sw2 = 0, np = 0;
  const int64_t e0 = (int64_t)blockIdx.x * kNoAllocRange;
  const int64_t e1 = e0 + kNoAllocRange < n ? e0 + kNoAllocRange : n;
  for (int64_t e = e0 + threadIdx.x; e < e1; e += 256) {
    const bool ok = pass ? pass[e] != 0 : true;
    if (ok) {
      const double w = (double)me2[e] * (double)wps[e] * wscale;
      sw += w;
      sw2 += w * w;
      np += 1.0;
    }
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    sw += __shfl_down_sync(0xffffffffu, sw, o);
    sw2 += __shfl_down_sync(0xffffffffu, sw2, o);
    np += __shfl_down_sync(0xffffffffu, np, o);
  }
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  if (lane == 0) {
    sh[0][w] = sw;
    sh[1][w] = sw2;
    sh[2][w] = np;
  }
  __syncthreads();
  if (threadIdx.x == 0) {
    double a = 0, b = 0, c = 0;
    for (int i = 0; i < 8; ++i) {
      a += sh[0][i];
      b += sh[1][i];
      c += sh[2][i];
    }
    partials[3 * blockIdx.x] = a;
    partials[3 * blockIdx.x + 1] = b;
    partials[3 * blockIdx.x + 2] = c;
  }
}
// finalize_kernel writing all four entries of acc to device memory (nb == 0: zeros)
__global__ void finalize_noalloc_kernel(const double* __restrict__ partials, int nb, int64_t n,
                                        double* __restrict__ acc) {
  __shared__ double sh[3][256];
  double a = 0, b = 0, c = 0;
  for (int i = threadIdx.x; i < nb; i += blockDim.x) {
    a += partials[3 * i];
    b += partials[3 * i + 1];
    c += partials[3 * i + 2];
  }
  sh[0][threadIdx.x] = a;
  sh[1][threadIdx.x] = b;
  sh[2][threadIdx.x] = c;
  __syncthreads();
  for (int s = blockDim.x / 2; s > 0; s >>= 1) {
    if ((int)threadIdx.x < s) {
      sh[0][threadIdx.x] += sh[0][threadIdx.x + s];
      sh[1][threadIdx.x] += sh[1][threadIdx.x + s];
      sh[2][threadIdx.x] += sh[2][threadIdx.x + s];
    }
    __syncthreads();
  }
  if (threadIdx.x == 0) {
    acc[0] = sh[0][0];
    acc[1] = sh[1][0];
    acc[2] = (double)n;
    acc[3] = sh[2][0];
  }
}

// Register-resident FMA chains: 8 independent accumulators per thread, `iters` x 8 FMAs each.
template <class T>
__global__ void __launch_bounds__(256) fma_peak_kernel(T* out, int iters, T a, T b) {
  T x0 = T(threadIdx.x) * T(1e-3), x1 = x0 + T(1), x2 = x0 + T(2), x3 = x0 + T(3), x4 = x0 + T(4),
    x5 = x0 + T(5), x6 = x0 + T(6), x7 = x0 + T(7);
  for (int i = 0; i < iters; ++i) {
#pragma unroll
    for (int r = 0; r < 8; ++r) {
      x0 = x0 * a + b;
      x1 = x1 * a + b;
      x2 = x2 * a + b;
      x3 = x3 * a + b;
      x4 = x4 * a + b;
      x5 = x5 * a + b;
      x6 = x6 * a + b;
      x7 = x7 * a + b;
    }
  }
  out[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = ((x0 + x1) + (x2 + x3)) + ((x4 + x5) + (x6 + x7));
}

// ---- adaptive grid: histograms of w^2 per (variable, bin)  (reading A22; role of the BASES grid-optimisation step)
//
// Deterministic, no atomics: block (b, s) takes slice s of the passing events of range b (the lists compact_kernel
// wrote for me_acc_kernel); inside a block every warp walks its share of the slice event by event with one LANE PER
// VARIABLE, so a lane owns row `lane` of the warp's private histogram in shared memory and nobody else touches it.
// The warps' histograms are added in warp order, the blocks' in block order (hist_finalize_kernel).
constexpr int kHistSplit = 4;      // blocks per range
constexpr int kHistWarps = 4;
constexpr int kHistMaxDim = 32;    // one lane per variable
__global__ void __launch_bounds__(32 * kHistWarps) hist_kernel(const uint8_t* __restrict__ bins,
                                                               const double* __restrict__ w,
                                                               const int* __restrict__ idx, const int* __restrict__ cnt,
                                                               int64_t m, int64_t range, int ndim, int nb,
                                                               double* __restrict__ partial) {
  extern __shared__ double hist_sh[];   // [kHistWarps][ndim][nb + 1]
  const int b = blockIdx.x / kHistSplit, sidx = blockIdx.x % kHistSplit;
  const int lane = threadIdx.x & 31, wp = threadIdx.x >> 5;
  const int row = nb + 1;
  for (int i = threadIdx.x; i < kHistWarps * ndim * row; i += blockDim.x) hist_sh[i] = 0.0;
  __syncthreads();
  const int total = cnt[b];
  const int per = (total + kHistSplit * kHistWarps - 1) / (kHistSplit * kHistWarps);
  const int lo = (sidx * kHistWarps + wp) * per;
  const int hi = lo + per < total ? lo + per : total;
  const int* __restrict__ my = idx + (int64_t)b * range;
  double* mine = hist_sh + ((size_t)wp * ndim + lane) * row;
  if (lane < ndim) {
    const uint8_t* __restrict__ brow = bins + (int64_t)lane * m;
    for (int j = lo; j < hi; ++j) {
      const int e = my[j];
      const double x = w[e];
      mine[brow[e]] += x * x;
    }
  }
  __syncthreads();
  double* out = partial + (size_t)blockIdx.x * ndim * nb;
  for (int i = threadIdx.x; i < ndim * nb; i += blockDim.x) {
    const int d = i / nb, k = i % nb;
    double a = 0.0;
    for (int q = 0; q < kHistWarps; ++q) a += hist_sh[((size_t)q * ndim + d) * row + k];
    out[i] = a;
  }
}

__global__ void hist_finalize_kernel(const double* __restrict__ partial, int nblk, int nel, double* __restrict__ hist) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= nel) return;
  double a = 0.0;
  for (int b = 0; b < nblk; ++b) a += partial[(size_t)b * nel + i];
  hist[i] += a;
}

cudaError_t GridAcc::launch(const uint8_t* d_bins, const double* d_w, const int* d_idx, const int* d_cnt, int64_t m,
                            int64_t range, int nblocks, int n_draws, cudaStream_t s) const {
  const int nblk = nblocks * kHistSplit;
  const size_t smem = sizeof(double) * kHistWarps * n_draws * (nb + 1);
  if (smem > 48 * 1024) {
    cudaError_t e = cudaFuncSetAttribute(hist_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
  }
  hist_kernel<<<nblk, 32 * kHistWarps, smem, s>>>(d_bins, d_w, d_idx, d_cnt, m, range, n_draws, nb, d_partial);
  const int nel = n_draws * nb;
  hist_finalize_kernel<<<(nel + 255) / 256, 256, 0, s>>>(d_partial, nblk, nel, d_hist);
  return cudaGetLastError();
}

// Makes the context's device current for the duration of a call and restores the caller's device afterwards
// (include/hg.h, hg_create): two contexts on different GPUs can be used from one thread.
struct DeviceGuard {
  int prev = -1;
  cudaError_t err = cudaSuccess;
  explicit DeviceGuard(int dev) {
    err = cudaGetDevice(&prev);
    if (err == cudaSuccess && prev != dev) err = cudaSetDevice(dev);
    else if (err == cudaSuccess) prev = -1;
  }
  ~DeviceGuard() {
    if (prev >= 0) cudaSetDevice(prev);
  }
};
#define HG_ON_DEVICE(ctx, who)                                              \
  DeviceGuard hg_guard((ctx)->device);                                      \
  if (hg_guard.err != cudaSuccess) return fail_cuda((ctx), hg_guard.err, who ": cudaSetDevice")

// sampling state of the context -> per-call constants
static void apply_sampling(const hg_ctx* ctx, PsConst& k) {
  k.grid = ctx->d_grid;
  k.nb = ctx->grid_nb;
  if (ctx->hadronic) {
    k.had = 1;
    k.y_res_max = ctx->had.y_res_max;
    for (int i = 0; i < 2; ++i) {
      k.pdf_norm[i] = ctx->had.pdf_norm[i];
      k.pdf_a[i] = ctx->had.pdf_a[i];
      k.pdf_b[i] = ctx->had.pdf_b[i];
    }
  }
}

// Global staging buffer of a process that stages in global memory (context-owned, grown on demand): sets *gblocks to
// the size of its persistent grid (0 for every other process).
static cudaError_t ensure_gstage(hg_ctx* ctx, const ProcVTable* vt, int precision, int* gblocks) {
  size_t bytes = 0;
  cudaError_t e = vt->gstage(precision, ctx->n_sm, gblocks, &bytes);
  if (e != cudaSuccess || bytes <= ctx->gstage_bytes) return e;
  if (ctx->d_gstage) cudaFree(ctx->d_gstage);
  ctx->d_gstage = nullptr;
  ctx->gstage_bytes = 0;
  e = cudaMalloc(&ctx->d_gstage, bytes);
  if (e == cudaSuccess) ctx->gstage_bytes = bytes;
  return e;
}

static bool misaligned(const void* p, size_t al) { return ((uintptr_t)p % al) != 0; }

static bool finite_pos(double x) { return isfinite(x) && x > 0.0; }
static bool finite_nonneg(double x) { return isfinite(x) && x >= 0.0; }

}  // namespace hg

using namespace hg;

extern "C" {

int hg_create(hg_ctx** out, int cuda_device) {
  if (!out) {
    g_create_error = "hg_create: out is NULL";
    return HG_EINVAL;
  }
  *out = nullptr;
  DeviceGuard guard(cuda_device);
  cudaError_t e = guard.err;
  if (e != cudaSuccess) {
    g_create_error = std::string("hg_create: cudaSetDevice: ") + cudaGetErrorString(e);
    return HG_ECUDA;
  }
  hg_ctx* ctx = new hg_ctx();
  ctx->device = cuda_device;
  cudaDeviceProp prop;
  e = cudaGetDeviceProperties(&prop, cuda_device);
  if (e == cudaSuccess) e = cudaMalloc(&ctx->d_partials, sizeof(double) * 3 * kMaxPartialBlocks);
  if (e == cudaSuccess) e = cudaMalloc(&ctx->d_acc, sizeof(double) * 3);
  if (e == cudaSuccess) e = cudaMallocHost(&ctx->h_acc, sizeof(double) * 3);
  if (e != cudaSuccess) {
    g_create_error = std::string("hg_create: ") + cudaGetErrorString(e);
    hg_destroy(ctx);
    return HG_ECUDA;
  }
  ctx->n_sm = prop.multiProcessorCount;
  for (int p = 1; p <= HG_N_PROCESS; ++p) default_cuts(p, &ctx->cuts[p]);
  *out = ctx;
  return HG_OK;
}

void hg_destroy(hg_ctx* ctx) {
  if (!ctx) return;
  DeviceGuard guard(ctx->device);
  if (ctx->d_partials) cudaFree(ctx->d_partials);
  if (ctx->d_acc) cudaFree(ctx->d_acc);
  if (ctx->h_acc) cudaFreeHost(ctx->h_acc);
  if (ctx->d_stage) cudaFree(ctx->d_stage);
  if (ctx->d_scratch) cudaFree(ctx->d_scratch);
  if (ctx->d_hist_partial) cudaFree(ctx->d_hist_partial);
  if (ctx->d_gstage) cudaFree(ctx->d_gstage);
  for (cudaEvent_t ev : ctx->ev) cudaEventDestroy(ev);
  for (int i = 0; i < 2; ++i) {
    if (ctx->ev_h2d[i]) cudaEventDestroy(ctx->ev_h2d[i]);
    if (ctx->ev_free[i]) cudaEventDestroy(ctx->ev_free[i]);
  }
  if (ctx->copy_stream) cudaStreamDestroy(ctx->copy_stream);
  delete ctx;
}

const char* hg_last_error(const hg_ctx* ctx) { return ctx ? ctx->err.c_str() : g_create_error.c_str(); }

void hg_default_params(hg_params* out) {
  if (out) default_params(out);
}

int hg_default_cuts(int process, hg_cuts* out) {
  if (!out) return HG_EINVAL;
  return default_cuts(process, out) ? HG_OK : HG_ENOPROC;
}

int hg_process_info(int process, hg_process_info_t* out) {
  if (!out) return HG_EINVAL;
  const ProcVTable* vt = vtable(process);
  if (!vt) return HG_ENOPROC;
  *out = vt->info;
  return HG_OK;
}

int hg_set_params(hg_ctx* ctx, const hg_params* par, const hg_cuts* cuts) {
  if (!ctx) return HG_EINVAL;
  if (!par) return fail(ctx, HG_EINVAL, "hg_set_params: par is NULL");
  if (!finite_pos(par->mz) || !finite_pos(par->mw) || !finite_pos(par->mt) || !finite_pos(par->alpha_em_inv) ||
      !finite_pos(par->alpha_s) || !finite_pos(par->mh))
    return fail(ctx, HG_EINVAL, "hg_set_params: masses and couplings must be finite and positive");
  if (!finite_pos(par->gz) || !finite_pos(par->gw) || !finite_pos(par->gt) || !finite_nonneg(par->gh))
    return fail(ctx, HG_EINVAL, "hg_set_params: widths must be finite and positive (Breit-Wigner mapping)");
  if (!finite_nonneg(par->mb)) return fail(ctx, HG_EINVAL, "hg_set_params: mb must be finite and >= 0");
  if (par->mb != 0.0) return fail(ctx, HG_EINVAL, "hg_set_params: only mb = 0 is generated (BASELINE.json)");
  if (!(par->mw < par->mz)) return fail(ctx, HG_EINVAL, "hg_set_params: need mw < mz (sw2 = 1 - mw^2/mz^2)");
  if (par->ckm_diagonal != 1) return fail(ctx, HG_EINVAL, "hg_set_params: only the diagonal CKM is implemented");
  if (par->complex_mass != 0 && par->complex_mass != 1)
    return fail(ctx, HG_EINVAL, "hg_set_params: complex_mass must be 0 or 1");
  if (cuts) {
    const double v[4] = {cuts->pt_jet_min, cuts->eta_jet_max, cuts->eta_lep_max, cuts->dr_jj_min};
    for (int i = 0; i < 4; ++i)
      if (!isfinite(v[i])) return fail(ctx, HG_EINVAL, "hg_set_params: cut values must be finite");
  }
  ctx->par = *par;
  ctx->coup = derive_couplings(*par);
  for (int p = 1; p <= HG_N_PROCESS; ++p) {
    if (cuts)
      ctx->cuts[p] = *cuts;
    else
      default_cuts(p, &ctx->cuts[p]);
  }
  ctx->params_set = true;
  return HG_OK;
}

// common argument checks; returns the vtable or NULL (code in *rc)
static const ProcVTable* check(hg_ctx* ctx, int process, int precision, int64_t n, int* rc, const char* who) {
  *rc = HG_OK;
  if (!ctx) {
    *rc = HG_EINVAL;
    return nullptr;
  }
  const ProcVTable* vt = vtable(process);
  if (!vt) {
    *rc = fail(ctx, HG_ENOPROC, (std::string(who) + ": unknown process id").c_str());
    return nullptr;
  }
  if (precision != HG_F64 && precision != HG_F32) {
    *rc = fail(ctx, HG_EINVAL, (std::string(who) + ": unknown precision").c_str());
    return nullptr;
  }
  if (n < 0) {
    *rc = fail(ctx, HG_EINVAL, (std::string(who) + ": n < 0").c_str());
    return nullptr;
  }
  if (!ctx->params_set) {
    *rc = fail(ctx, HG_ENOTSET, (std::string(who) + ": hg_set_params has not been called").c_str());
    return nullptr;
  }
  return vt;
}

static int check_rs(hg_ctx* ctx, const ProcVTable* vt, int process, double rs, const char* who) {
  if (!finite_pos(rs)) return fail(ctx, HG_EINVAL, (std::string(who) + ": sqrt_s_hat must be finite and > 0").c_str());
  if (ctx->hadronic) {
    if (!vt->has_hadronic())
      return fail(ctx, HG_EINVAL, (std::string(who) + ": the hadronic phase space is not implemented for this process").c_str());
    const double ptmin = ctx->cuts[process].pt_jet_min > 0 ? ctx->cuts[process].pt_jet_min : 1.0;
    if (!(2.0 * ptmin < rs)) return fail(ctx, HG_EINVAL, (std::string(who) + ": sqrt(s) below twice the jet pT cut").c_str());
    return HG_OK;
  }
  if (process == HG_GG_TTXG_DILEP) {
    // the Breit-Wigner windows must always be kinematically open (reading A14): no rejection on the device
    const double mtmax = sqrt(ctx->par.mt * ctx->par.mt + ctx->par.mt * ctx->par.gt * fmin(20.0, ctx->par.mt / ctx->par.gt));
    const double mwmax = sqrt(ctx->par.mw * ctx->par.mw + ctx->par.mw * ctx->par.gw * fmin(20.0, ctx->par.mw / ctx->par.gw));
    const double mtmin2 = ctx->par.mt * ctx->par.mt - ctx->par.mt * ctx->par.gt * fmin(20.0, ctx->par.mt / ctx->par.gt);
    if (!(2.0 * mtmax < rs) || !(mtmin2 > 0) || !(mwmax < sqrt(mtmin2)))
      return fail(ctx, HG_EINVAL, (std::string(who) + ": Breit-Wigner windows not open at this sqrt_s_hat").c_str());
  }
  // massive final states: the threshold must be open
  double msum = 0.0;
  if (process == HG_UDX_EPVEH) msum = ctx->par.mh;
  if (process == HG_UUX_EPEMHH) msum = 2.0 * ctx->par.mh;
  if (process == HG_GG_TTXH) msum = 2.0 * ctx->par.mt + ctx->par.mh;
  if (process == HG_UD_HUD) msum = ctx->par.mh;
  if (process == HG_UD_HHUD) msum = 2.0 * ctx->par.mh;
  if (!(msum < rs)) return fail(ctx, HG_EINVAL, (std::string(who) + ": sqrt_s_hat is below the threshold").c_str());
  (void)vt;
  return HG_OK;
}

int hg_gen_phase_space(hg_ctx* ctx, int process, int precision, uint64_t seed, uint64_t first_event, int64_t n,
                       double sqrt_s_hat, void* d_p, void* d_wps, uint8_t* d_pass, void* cuda_stream) {
  int rc;
  const ProcVTable* vt = check(ctx, process, precision, n, &rc, "hg_gen_phase_space");
  if (!vt) return rc;
  if ((rc = check_rs(ctx, vt, process, sqrt_s_hat, "hg_gen_phase_space")) != HG_OK) return rc;
  if (ctx->d_grid && ctx->grid_ndim != vt->info.n_draws)
    return fail(ctx, HG_EINVAL, "hg_gen_phase_space: the grid set by hg_set_grid has another number of draws than this process");
  if (n == 0) return HG_OK;
  if (!d_p || !d_wps) return fail(ctx, HG_EINVAL, "hg_gen_phase_space: d_p / d_wps is NULL");
  if (misaligned(d_p, precision == HG_F64 ? 8 : 4) || misaligned(d_wps, precision == HG_F64 ? 8 : 4))
    return fail(ctx, HG_EINVAL, "hg_gen_phase_space: misaligned pointer");
  HG_ON_DEVICE(ctx, "hg_gen_phase_space");
  const int n_rambo = process == HG_GG_TTXG_DILEP ? 3 : vt->info.n_final;
  PsConst k = make_psconst(ctx->par, ctx->cuts[process], n_rambo, sqrt_s_hat);
  apply_sampling(ctx, k);
  cudaError_t e = vt->ps(precision, n, k, seed, first_event, d_p, d_wps, d_pass, (cudaStream_t)cuda_stream);
  if (e != cudaSuccess) return fail_cuda(ctx, e, "hg_gen_phase_space");
  return HG_OK;
}

int hg_matrix_element(hg_ctx* ctx, int process, int precision, int64_t n, const void* d_p, void* d_me2,
                      void* cuda_stream) {
  int rc;
  const ProcVTable* vt = check(ctx, process, precision, n, &rc, "hg_matrix_element");
  if (!vt) return rc;
  if (n == 0) return HG_OK;
  if (!d_p || !d_me2) return fail(ctx, HG_EINVAL, "hg_matrix_element: d_p / d_me2 is NULL");
  const size_t al = precision == HG_F64 ? 8 : 4;
  if (((uintptr_t)d_p % al) || ((uintptr_t)d_me2 % al))
    return fail(ctx, HG_EINVAL, "hg_matrix_element: misaligned pointer");
  HG_ON_DEVICE(ctx, "hg_matrix_element");
  int gblocks = 0;
  cudaError_t e = ensure_gstage(ctx, vt, precision, &gblocks);
  if (e != cudaSuccess) return fail_cuda(ctx, e, "hg_matrix_element: global staging buffer");
  e = vt->me(precision, n, d_p, d_me2, ctx->coup, ctx->d_gstage, gblocks, 0.0, (cudaStream_t)cuda_stream);
  if (e != cudaSuccess) return fail_cuda(ctx, e, "hg_matrix_element");
  return HG_OK;
}

// sqrt_s_hat > 0: h_p holds the final-state legs only (hg_matrix_element_host_cm)
static int me_host(hg_ctx* ctx, int process, int precision, int64_t n, double sqrt_s_hat, const void* h_p,
                   void* h_me2, void* cuda_stream) {
  int rc;
  const ProcVTable* vt = check(ctx, process, precision, n, &rc, "hg_matrix_element_host");
  if (!vt) return rc;
  if (n == 0) return HG_OK;
  if (!h_p || !h_me2) return fail(ctx, HG_EINVAL, "hg_matrix_element_host: h_p / h_me2 is NULL");
  if (misaligned(h_p, precision == HG_F64 ? 8 : 4) || misaligned(h_me2, precision == HG_F64 ? 8 : 4))
    return fail(ctx, HG_EINVAL, "hg_matrix_element_host: misaligned pointer");
  HG_ON_DEVICE(ctx, "hg_matrix_element_host");
  // Pipelined in chunks of kHostChunk events over two device buffers: the H2D copy of chunk i+1 (on a context-owned
  // copy stream) overlaps the kernel and the D2H copy of chunk i (on the caller's stream).  The host array is
  // [n_ext][4][n], so one chunk is 4 n_ext strided rows: one cudaMemcpy2DAsync.
  const size_t el = precision == HG_F64 ? 8 : 4;
  const int rows = 4 * (sqrt_s_hat > 0.0 ? vt->info.n_ext - 2 : vt->info.n_ext);
  const int64_t chunk = n < kHostChunk ? n : kHostChunk;
  const size_t in_bytes = el * rows * (size_t)chunk, out_bytes = el * (size_t)chunk;
  const size_t buf_bytes = (in_bytes + out_bytes + 255) / 256 * 256;
  if (ctx->stage_bytes < 2 * buf_bytes) {
    if (ctx->d_stage) cudaFree(ctx->d_stage);
    ctx->d_stage = nullptr;
    ctx->stage_bytes = 0;
    cudaError_t e = cudaMalloc(&ctx->d_stage, 2 * buf_bytes);
    if (e != cudaSuccess) return fail_cuda(ctx, e, "hg_matrix_element_host: cudaMalloc");
    ctx->stage_bytes = 2 * buf_bytes;
  }
  int gblocks = 0;
  cudaError_t e = ensure_gstage(ctx, vt, precision, &gblocks);
  if (e != cudaSuccess) return fail_cuda(ctx, e, "hg_matrix_element_host: global staging buffer");
  if (!ctx->copy_stream) {
    e = cudaStreamCreateWithFlags(&ctx->copy_stream, cudaStreamNonBlocking);
    for (int i = 0; i < 2 && e == cudaSuccess; ++i) {
      e = cudaEventCreateWithFlags(&ctx->ev_h2d[i], cudaEventDisableTiming);
      if (e == cudaSuccess) e = cudaEventCreateWithFlags(&ctx->ev_free[i], cudaEventDisableTiming);
    }
    if (e != cudaSuccess) return fail_cuda(ctx, e, "hg_matrix_element_host: stream/event creation");
  }
  cudaStream_t s = (cudaStream_t)cuda_stream;
  // the copy stream must not start before work already queued on the caller's stream that uses the buffers
  e = cudaEventRecord(ctx->ev_free[0], s);
  if (e == cudaSuccess) e = cudaEventRecord(ctx->ev_free[1], s);
  int i = 0;
  for (int64_t off = 0; off < n && e == cudaSuccess; off += chunk, ++i) {
    const int64_t m = n - off < chunk ? n - off : chunk;
    const int b = i & 1;
    char* d_in = (char*)ctx->d_stage + (size_t)b * buf_bytes;
    char* d_out = d_in + in_bytes;
    e = cudaStreamWaitEvent(ctx->copy_stream, ctx->ev_free[b], 0);   // buffer b no longer read by chunk i-2
    if (e == cudaSuccess)
      e = cudaMemcpy2DAsync(d_in, el * (size_t)m, (const char*)h_p + el * (size_t)off, el * (size_t)n,
                            el * (size_t)m, rows, cudaMemcpyHostToDevice, ctx->copy_stream);
    if (e == cudaSuccess) e = cudaEventRecord(ctx->ev_h2d[b], ctx->copy_stream);
    if (e == cudaSuccess) e = cudaStreamWaitEvent(s, ctx->ev_h2d[b], 0);
    if (e == cudaSuccess)
      e = vt->me(precision, m, d_in, d_out, ctx->coup, ctx->d_gstage, gblocks, 0.5 * sqrt_s_hat, s);
    if (e == cudaSuccess)
      e = cudaMemcpyAsync((char*)h_me2 + el * (size_t)off, d_out, el * (size_t)m, cudaMemcpyDeviceToHost, s);
    if (e == cudaSuccess) e = cudaEventRecord(ctx->ev_free[b], s);
  }
  if (e == cudaSuccess) e = cudaStreamSynchronize(s);
  if (e != cudaSuccess) return fail_cuda(ctx, e, "hg_matrix_element_host");
  return HG_OK;
}

int hg_matrix_element_host(hg_ctx* ctx, int process, int precision, int64_t n, const void* h_p, void* h_me2,
                           void* cuda_stream) {
  return me_host(ctx, process, precision, n, 0.0, h_p, h_me2, cuda_stream);
}

int hg_matrix_element_host_cm(hg_ctx* ctx, int process, int precision, int64_t n, double sqrt_s_hat,
                              const void* h_pfinal, void* h_me2, void* cuda_stream) {
  if (!ctx) return HG_EINVAL;
  if (!finite_pos(sqrt_s_hat))
    return fail(ctx, HG_EINVAL, "hg_matrix_element_host_cm: sqrt_s_hat must be finite and > 0");
  return me_host(ctx, process, precision, n, sqrt_s_hat, h_pfinal, h_me2, cuda_stream);
}

// finalize partials -> acc (host), synchronising the stream
static int finish(hg_ctx* ctx, int nblocks, int64_t n, double acc[4], cudaStream_t s, const char* who) {
  finalize_kernel<<<1, 256, 0, s>>>(ctx->d_partials, nblocks, ctx->d_acc);
  cudaError_t e = cudaGetLastError();
  if (e == cudaSuccess) e = cudaMemcpyAsync(ctx->h_acc, ctx->d_acc, 3 * sizeof(double), cudaMemcpyDeviceToHost, s);
  if (e == cudaSuccess) e = cudaStreamSynchronize(s);
  if (e != cudaSuccess) return fail_cuda(ctx, e, who);
  acc[0] = ctx->h_acc[0];
  acc[1] = ctx->h_acc[1];
  acc[2] = (double)n;
  acc[3] = ctx->h_acc[2];
  return HG_OK;
}

int hg_accumulate(hg_ctx* ctx, int precision, int64_t n, const void* d_me2, const void* d_wps,
                  const uint8_t* d_pass, double sqrt_s_hat, double acc[4], void* cuda_stream) {
  if (!ctx) return HG_EINVAL;
  if (precision != HG_F64 && precision != HG_F32) return fail(ctx, HG_EINVAL, "hg_accumulate: unknown precision");
  if (n < 0) return fail(ctx, HG_EINVAL, "hg_accumulate: n < 0");
  if (!acc) return fail(ctx, HG_EINVAL, "hg_accumulate: acc is NULL");
  if (!finite_pos(sqrt_s_hat)) return fail(ctx, HG_EINVAL, "hg_accumulate: sqrt_s_hat must be finite and > 0");
  acc[0] = acc[1] = acc[2] = acc[3] = 0.0;
  if (n == 0) return HG_OK;
  if (!d_me2 || !d_wps) return fail(ctx, HG_EINVAL, "hg_accumulate: d_me2 / d_wps is NULL");
  if (misaligned(d_me2, precision == HG_F64 ? 8 : 4) || misaligned(d_wps, precision == HG_F64 ? 8 : 4))
    return fail(ctx, HG_EINVAL, "hg_accumulate: misaligned pointer");
  HG_ON_DEVICE(ctx, "hg_accumulate");
  cudaStream_t s = (cudaStream_t)cuda_stream;
  const double wscale = kHbarC2Pb / (2.0 * sqrt_s_hat * sqrt_s_hat);
  int nblocks = ctx->n_sm * 8;
  if (nblocks > kMaxPartialBlocks) nblocks = kMaxPartialBlocks;
  const int64_t need = (n + 255) / 256;
  if (need < nblocks) nblocks = (int)need;
  if (precision == HG_F64)
    accumulate_kernel<double><<<nblocks, 256, 0, s>>>((const double*)d_me2, (const double*)d_wps, d_pass, n, wscale,
                                                      ctx->d_partials);
  else
    accumulate_kernel<float><<<nblocks, 256, 0, s>>>((const float*)d_me2, (const float*)d_wps, d_pass, n, wscale,
                                                     ctx->d_partials);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return fail_cuda(ctx, e, "hg_accumulate");
  return finish(ctx, nblocks, n, acc, s, "hg_accumulate");
}

// Device address of hg_noalloc_partials on the current device: looked up once per device, with that device
// current (the symbol has one instance per device).  No allocation.
static int noalloc_scratch(double** out) {
  static std::mutex mu;
  static double* ptr[kNoAllocMaxDevices] = {};
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return fail_cuda_noctx(e, "hg_accumulate_noalloc: cudaGetDevice");
  if (dev < 0 || dev >= kNoAllocMaxDevices) return fail_noctx(HG_EINVAL, "hg_accumulate_noalloc: device index out of range");
  std::lock_guard<std::mutex> lock(mu);
  if (!ptr[dev]) {
    double* p = nullptr;
    e = cudaGetSymbolAddress((void**)&p, hg_noalloc_partials);
    if (e != cudaSuccess) return fail_cuda_noctx(e, "hg_accumulate_noalloc: cudaGetSymbolAddress");
    if (!p) return fail_noctx(HG_ECUDA, "hg_accumulate_noalloc: cudaGetSymbolAddress returned NULL");
    ptr[dev] = p;
  }
  *out = ptr[dev];
  return HG_OK;
}

int hg_accumulate_noalloc(int precision, int64_t n, const void* d_me2, const void* d_wps, const uint8_t* d_pass,
                          double sqrt_s_hat, double* d_acc, void* cuda_stream) {
  if (precision != HG_F64 && precision != HG_F32) return fail_noctx(HG_EINVAL, "hg_accumulate_noalloc: unknown precision");
  if (n < 0) return fail_noctx(HG_EINVAL, "hg_accumulate_noalloc: n < 0");
  if (n > (int64_t)HG_NOALLOC_MAX_EVENTS)
    return fail_noctx(HG_EINVAL, "hg_accumulate_noalloc: n exceeds HG_NOALLOC_MAX_EVENTS (16777216 events: the static "
                                 "scratch array holds 4096 blocks of 4096 events); split the batch");
  if (!d_acc) return fail_noctx(HG_EINVAL, "hg_accumulate_noalloc: d_acc is NULL");
  if (misaligned(d_acc, 8)) return fail_noctx(HG_EINVAL, "hg_accumulate_noalloc: misaligned d_acc");
  if (!finite_pos(sqrt_s_hat)) return fail_noctx(HG_EINVAL, "hg_accumulate_noalloc: sqrt_s_hat must be finite and > 0");
  if (n > 0 && (!d_me2 || !d_wps)) return fail_noctx(HG_EINVAL, "hg_accumulate_noalloc: d_me2 / d_wps is NULL");
  if (misaligned(d_me2, precision == HG_F64 ? 8 : 4) || misaligned(d_wps, precision == HG_F64 ? 8 : 4))
    return fail_noctx(HG_EINVAL, "hg_accumulate_noalloc: misaligned pointer");
  double* scratch = nullptr;
  const int rc = noalloc_scratch(&scratch);
  if (rc != HG_OK) return rc;
  cudaStream_t s = (cudaStream_t)cuda_stream;
  const double wscale = kHbarC2Pb / (2.0 * sqrt_s_hat * sqrt_s_hat);
  const int nblocks = (int)((n + kNoAllocRange - 1) / kNoAllocRange);   // <= kNoAllocMaxBlocks
  if (nblocks > 0) {
    if (precision == HG_F64)
      accumulate_noalloc_kernel<double><<<nblocks, 256, 0, s>>>((const double*)d_me2, (const double*)d_wps, d_pass, n,
                                                                wscale, scratch);
    else
      accumulate_noalloc_kernel<float><<<nblocks, 256, 0, s>>>((const float*)d_me2, (const float*)d_wps, d_pass, n,
                                                               wscale, scratch);
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail_cuda_noctx(e, "hg_accumulate_noalloc: accumulate_noalloc_kernel");
  }
  finalize_noalloc_kernel<<<1, 256, 0, s>>>(scratch, nblocks, n, d_acc);
  const cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return fail_cuda_noctx(e, "hg_accumulate_noalloc: finalize_noalloc_kernel");
  return HG_OK;
}

int hg_integrate_step(hg_ctx* ctx, int process, int precision, uint64_t seed, uint64_t first_event, int64_t n,
                      double sqrt_s_hat, double acc[4], void* cuda_stream) {
  int rc;
  const ProcVTable* vt = check(ctx, process, precision, n, &rc, "hg_integrate_step");
  if (!vt) return rc;
  if (!acc) return fail(ctx, HG_EINVAL, "hg_integrate_step: acc is NULL");
  if ((rc = check_rs(ctx, vt, process, sqrt_s_hat, "hg_integrate_step")) != HG_OK) return rc;
  if (ctx->d_grid && ctx->grid_ndim != vt->info.n_draws)
    return fail(ctx, HG_EINVAL, "hg_integrate_step: the grid set by hg_set_grid has another number of draws than this process");
  acc[0] = acc[1] = acc[2] = acc[3] = 0.0;
  if (n == 0) return HG_OK;
  HG_ON_DEVICE(ctx, "hg_integrate_step");
  cudaStream_t s = (cudaStream_t)cuda_stream;
  const int n_rambo = process == HG_GG_TTXG_DILEP ? 3 : vt->info.n_final;
  PsConst k = make_psconst(ctx->par, ctx->cuts[process], n_rambo, sqrt_s_hat);
  apply_sampling(ctx, k);
  const bool hist = ctx->d_grid && ctx->d_hist;      // grid-optimisation step: accumulate the histograms
  const bool split = vt->split_step() || ctx->d_grid != nullptr || ctx->hadronic;   // grid / hadronic: split step
  const double wscale = kHbarC2Pb / (2.0 * sqrt_s_hat * sqrt_s_hat);
  int per_sm = 1;
  cudaError_t e = vt->int_blocks_per_sm(precision, split, &per_sm);
  if (e != cudaSuccess) return fail_cuda(ctx, e, "hg_integrate_step: occupancy query");
  if (per_sm < 1) per_sm = 1;
  int nblocks = ctx->n_sm * per_sm;  // persistent grid: a whole number of resident waves
  if (nblocks > kMaxPartialBlocks) nblocks = kMaxPartialBlocks;
  int gblocks = 0;
  e = ensure_gstage(ctx, vt, precision, &gblocks);
  if (e != cudaSuccess) return fail_cuda(ctx, e, "hg_integrate_step: global staging buffer");
  if (gblocks > 0 && nblocks > gblocks) nblocks = gblocks;
  const int64_t need = (n + kIntThreads - 1) / kIntThreads;
  if (need < nblocks) nblocks = (int)need;
  const int64_t chunk = n < kIntChunk ? n : kIntChunk;
  const bool per_event = split;
  if (split) {  // separate kernels per chunk through a context-owned buffer, grown on demand
    const size_t bytes = vt->scratch_bytes(precision, chunk, hist);
    if (bytes > ctx->scratch_bytes) {
      if (ctx->d_scratch) cudaFree(ctx->d_scratch);
      ctx->d_scratch = nullptr;
      ctx->scratch_bytes = 0;
      e = cudaMalloc(&ctx->d_scratch, bytes);
      if (e != cudaSuccess) return fail_cuda(ctx, e, "hg_integrate_step: cudaMalloc of the chunk buffer");
      ctx->scratch_bytes = bytes;
    }
  }
  GridAcc ga;
  if (hist) {
    const size_t bytes = sizeof(double) * (size_t)nblocks * kHistSplit * vt->info.n_draws * ctx->grid_nb;
    if (bytes > ctx->hist_partial_bytes) {
      if (ctx->d_hist_partial) cudaFree(ctx->d_hist_partial);
      ctx->d_hist_partial = nullptr;
      ctx->hist_partial_bytes = 0;
      e = cudaMalloc(&ctx->d_hist_partial, bytes);
      if (e != cudaSuccess) return fail_cuda(ctx, e, "hg_integrate_step: cudaMalloc of the histogram partials");
      ctx->hist_partial_bytes = bytes;
    }
    ga.nb = ctx->grid_nb;
    ga.d_partial = ctx->d_hist_partial;
    ga.d_hist = ctx->d_hist;
  }
  const int nchunks = per_event ? (int)((n + chunk - 1) / chunk) : 1;
  cudaEvent_t* ev = nullptr;
  if (ctx->profiling) {
    while ((int)ctx->ev.size() < 3 * nchunks) {
      cudaEvent_t x;
      if ((e = cudaEventCreate(&x)) != cudaSuccess) return fail_cuda(ctx, e, "hg_integrate_step: cudaEventCreate");
      ctx->ev.push_back(x);
    }
    ev = ctx->ev.data();
  }
  e = vt->integrate(precision, n, k, seed, first_event, ctx->coup, wscale, ctx->d_partials, nblocks, ctx->d_scratch,
                    chunk, ev, hist ? &ga : nullptr, ctx->d_gstage, s);
  if (e != cudaSuccess) return fail_cuda(ctx, e, "hg_integrate_step");
  ctx->n_launches = (per_event ? (hist ? 5 : 3) * nchunks : 1) + 1;
  rc = finish(ctx, nblocks, n, acc, s, "hg_integrate_step");  // synchronises the stream
  if (rc == HG_OK && ev) {
    ctx->t_ps_ms = ctx->t_me_ms = 0;
    for (int i = 0; i < nchunks; ++i) {
      float a = 0, b = 0;
      if (per_event) {
        cudaEventElapsedTime(&a, ev[3 * i], ev[3 * i + 1]);
        cudaEventElapsedTime(&b, ev[3 * i + 1], ev[3 * i + 2]);
      } else {
        cudaEventElapsedTime(&b, ev[0], ev[2]);
      }
      ctx->t_ps_ms += a;
      ctx->t_me_ms += b;
    }
  }
  return rc;
}

int hg_default_hadronic(int process, hg_hadronic* out) {
  if (!out) return HG_EINVAL;
  return default_hadronic(process, out) ? HG_OK : HG_ENOPROC;
}

int hg_set_hadronic(hg_ctx* ctx, const hg_hadronic* h) {
  if (!ctx) return HG_EINVAL;
  if (!h) {
    ctx->hadronic = false;
    return HG_OK;
  }
  if (!finite_pos(h->y_res_max)) return fail(ctx, HG_EINVAL, "hg_set_hadronic: y_res_max must be finite and > 0");
  for (int i = 0; i < 2; ++i)
    if (!finite_nonneg(h->pdf_norm[i]) || !isfinite(h->pdf_a[i]) || !finite_nonneg(h->pdf_b[i]))
      return fail(ctx, HG_EINVAL, "hg_set_hadronic: parton-density parameters must be finite, norm and b >= 0");
  ctx->had = *h;
  ctx->hadronic = true;
  return HG_OK;
}

int hg_set_grid(hg_ctx* ctx, const double* d_grid, int n_dim, int n_bins, double* d_hist) {
  if (!ctx) return HG_EINVAL;
  if (!d_grid) {
    ctx->d_grid = nullptr;
    ctx->grid_nb = ctx->grid_ndim = 0;
    ctx->d_hist = nullptr;
    return HG_OK;
  }
  if (n_bins < 2 || n_bins > HG_GRID_MAX_BINS) return fail(ctx, HG_EINVAL, "hg_set_grid: n_bins out of range");
  if (n_dim < 1 || n_dim > kHistMaxDim) return fail(ctx, HG_EINVAL, "hg_set_grid: n_dim out of range");
  if (misaligned(d_grid, 8) || misaligned(d_hist, 8)) return fail(ctx, HG_EINVAL, "hg_set_grid: misaligned pointer");
  ctx->d_grid = d_grid;
  ctx->grid_nb = n_bins;
  ctx->grid_ndim = n_dim;
  ctx->d_hist = d_hist;
  return HG_OK;
}

int hg_grid_refine(int n_dim, int n_bins, const double* h_hist, double alpha, double* h_grid) {
  if (n_dim < 1 || n_bins < 2 || n_bins > HG_GRID_MAX_BINS || !h_hist || !h_grid || !(alpha >= 0.0)) return HG_EINVAL;
  const int nb = n_bins;
  std::vector<double> sm(nb), r(nb), edges(nb + 1);
  for (int d = 0; d < n_dim; ++d) {
    const double* h = h_hist + (size_t)d * nb;
    double* g = h_grid + (size_t)d * (nb + 1);
    double tot = 0.0;
    bool fin = true;
    for (int i = 0; i < nb; ++i) {
      fin = fin && isfinite(h[i]);
      tot += h[i];
    }
    if (!fin || !(tot > 0.0)) continue;            // nothing accumulated for this variable: grid unchanged
    // smoothing over neighbouring bins, normalisation
    sm[0] = (h[0] + h[1]) / 2.0;
    sm[nb - 1] = (h[nb - 2] + h[nb - 1]) / 2.0;
    for (int i = 1; i < nb - 1; ++i) sm[i] = (h[i - 1] + h[i] + h[i + 1]) / 3.0;
    double ssum = 0.0;
    for (int i = 0; i < nb; ++i) ssum += sm[i];
    // compression r = ((1 - s) / ln(1 / s))^alpha
    double rsum = 0.0;
    for (int i = 0; i < nb; ++i) {
      const double x = sm[i] / ssum;
      r[i] = 0.0;
      if (x > 0.0) r[i] = x >= 1.0 ? 1.0 : pow((1.0 - x) / log(1.0 / x), alpha);
      rsum += r[i];
    }
    const double per = rsum / nb;
    if (!(per > 0.0)) continue;
    // new edges: every new bin holds `per`, r spread evenly inside an old bin
    edges[0] = 0.0;
    edges[nb] = 1.0;
    int k = 0;
    double acc = 0.0;
    for (int j = 1; j < nb; ++j) {
      const double target = j * per;
      while (k < nb - 1 && acc + r[k] < target) {
        acc += r[k];
        ++k;
      }
      double frac = r[k] > 0.0 ? (target - acc) / r[k] : 0.0;
      frac = frac < 0.0 ? 0.0 : (frac > 1.0 ? 1.0 : frac);
      edges[j] = g[k] + frac * (g[k + 1] - g[k]);
    }
    for (int j = 1; j <= nb; ++j)
      if (!(edges[j] > edges[j - 1])) edges[j] = nextafter(edges[j - 1], 2.0);
    edges[nb] = 1.0;
    for (int j = 0; j <= nb; ++j) g[j] = edges[j];
  }
  return HG_OK;
}

int hg_set_profiling(hg_ctx* ctx, int on) {
  if (!ctx) return HG_EINVAL;
  ctx->profiling = on ? 1 : 0;
  return HG_OK;
}

int hg_last_step_info(const hg_ctx* ctx, double out[3]) {
  if (!ctx || !out) return HG_EINVAL;
  out[0] = ctx->t_ps_ms;
  out[1] = ctx->t_me_ms;
  out[2] = (double)ctx->n_launches;
  return HG_OK;
}

int hg_measure_fma_peak(hg_ctx* ctx, int precision, double* flops_per_s, void* cuda_stream) {
  if (!ctx) return HG_EINVAL;
  if (!flops_per_s) return fail(ctx, HG_EINVAL, "hg_measure_fma_peak: flops_per_s is NULL");
  if (precision != HG_F64 && precision != HG_F32) return fail(ctx, HG_EINVAL, "hg_measure_fma_peak: unknown precision");
  HG_ON_DEVICE(ctx, "hg_measure_fma_peak");
  cudaStream_t s = (cudaStream_t)cuda_stream;
  const int blocks = ctx->n_sm * 8, threads = 256, iters = precision == HG_F64 ? 4096 : 8192;
  void* d_out = nullptr;
  cudaError_t e = cudaMalloc(&d_out, (size_t)blocks * threads * 8);
  if (e != cudaSuccess) return fail_cuda(ctx, e, "hg_measure_fma_peak: cudaMalloc");
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0);
  cudaEventCreate(&e1);
  float best = 1e30f;
  for (int rep = 0; rep < 6 && e == cudaSuccess; ++rep) {
    cudaEventRecord(e0, s);
    if (precision == HG_F64)
      fma_peak_kernel<double><<<blocks, threads, 0, s>>>((double*)d_out, iters, 0.999999, 1e-6);
    else
      fma_peak_kernel<float><<<blocks, threads, 0, s>>>((float*)d_out, iters, 0.99999f, 1e-5f);
    cudaEventRecord(e1, s);
    e = cudaEventSynchronize(e1);
    float ms = 0;
    if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
    if (rep > 0 && ms < best) best = ms;
  }
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  cudaFree(d_out);
  if (e != cudaSuccess) return fail_cuda(ctx, e, "hg_measure_fma_peak");
  const double flops = 2.0 * 64.0 * (double)iters * (double)blocks * (double)threads;
  *flops_per_s = flops / ((double)best * 1e-3);
  return HG_OK;
}

}  // extern "C"
