/* hg.h -- C ABI of the B200 tree-level |M|^2 library (libhg.so).
 *
 * The hot path of arXiv:1305.0708 ("Fast computation of MadGraph amplitudes on GPU"): for a batch of
 * phase-space points, evaluate the tree-level Standard Model matrix element squared, summed over
 * helicities and colours and averaged over the initial state (Eq. 4-6), multiply by the
 * phase-space weight and flux factor, and accumulate a Monte-Carlo cross section.
 *
 * Conventions common to every call
 *   - units GeV, metric (+,-,-,-); momenta are physical (E > 0) for every external leg;
 *   - "d_" pointers are DEVICE memory owned by the caller (the library never allocates per call and never
 *     frees caller memory); "h_" pointers are HOST memory owned by the caller;
 *   - momenta layout is structure-of-arrays p[leg][mu][event]: element (leg l, component mu, event e) sits
 *     at index (l*4 + mu)*n + e; mu = 0..3 = (E, px, py, pz); leg order = initial then final state as
 *     listed under hg_process below;
 *   - precision HG_F64: every d_ array is double; HG_F32: every d_ array is float (accumulators stay
 *     double);
 *   - cuda_stream is a cudaStream_t passed as void* (NULL = default stream); calls are asynchronous on it
 *     unless stated otherwise;
 *   - every call returns 0 on success or a negative hg_status; the message of the last failure of a
 *     context is available from hg_last_error().  Nothing throws across the ABI.  Arguments are validated
 *     before any launch (NULL or misaligned pointers, n < 0, unknown process/precision, parameters not set).  n == 0 is
 *     a successful no-op.
 *   - results depend only on (params, cuts, process, precision, seed, first_event, n, sqrt_s_hat): event
 *     k always uses Philox counter k (reading SURVEY.md 8c-A15), so batches can be split or sharded.
 */
#ifndef HG_H
#define HG_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct hg_ctx hg_ctx; /* opaque, library-owned */

enum hg_status {
  HG_OK = 0,
  HG_EINVAL = -1,  /* bad argument */
  HG_ENOPROC = -2, /* unknown process id */
  HG_ECUDA = -3,   /* CUDA runtime error (text in hg_last_error) */
  HG_ENOTSET = -4  /* hg_set_params has not been called on this context */
};

enum hg_precision { HG_F64 = 0, HG_F32 = 1 };

/* The five BASELINE.json configs (workloads of PAPER.md:147-256, Eq. 12a, 13a, 17d).  Leg order:
 *   HG_UDX_EPVE      u d~ -> e+ ve                                  (4 legs)
 *   HG_UUX_EPEMG     u u~ -> e+ e- g                                (5 legs)
 *   HG_UDX_EPVEGG    u d~ -> e+ ve g g                              (6 legs)
 *   HG_GG_TTXG_DILEP g g  -> b e+ ve b~ mu- vm~ g   via t t~ g       (9 legs; decay-chain diagrams only)
 *   HG_UDX_EPVEGGG   u d~ -> e+ ve g g g                            (7 legs)                         */
enum hg_process {
  HG_UDX_EPVE = 1,
  HG_UUX_EPEMG = 2,
  HG_UDX_EPVEGG = 3,
  HG_GG_TTXG_DILEP = 4,
  HG_UDX_EPVEGGG = 5,
  /* Higgs-sector processes: exercise the FFS, VVS, VVSS and SSS vertices of the library
   * (Eq. 39, 50-52); no cuts, massive final states from massive RAMBO.
   *   HG_UDX_EPVEH   u d~ -> e+ ve h      (5 legs)  W* -> W H
   *   HG_UUX_EPEMHH  u u~ -> e+ e- h h    (6 legs)  Z* -> Z H H: Z Z H twice, Z Z H H, H H H
   *   HG_GG_TTXH     g g -> t t~ h        (5 legs)  t t H Yukawa on massive external tops (Eq. 20d) */
  HG_UDX_EPVEH = 6,
  HG_UUX_EPEMHH = 7,
  HG_GG_TTXH = 8,
  /* next size up: u d~ -> e+ ve g g g g, 8 legs, 428 Feynman diagrams / 516
   * colour-split amplitudes, 24 colour flows, 16 of 256 helicity combinations non-zero; cuts as config 5 */
  HG_UDX_EPVEGGGG = 9,
  /* weak-boson fusion (Eq. 21a, 22a): two quark lines, W W and Z Z
   * fusion with their interference (two colour flows, relative Fermi sign); no cuts; massive RAMBO.
   *   HG_UD_HUD    u d -> h u d      (5 legs)  W W H, Z Z H
   *   HG_UD_HHUD   u d -> h h u d    (6 legs)  + W W H H, Z Z H H, H H H */
  HG_UD_HUD = 10,
  HG_UD_HHUD = 11
};
#define HG_N_PROCESS 11
#define HG_MAX_EXT 9

/* Standard Model inputs (paper's own: PAPER.md:1075; the configs override them).
 * Derived inside hg_set_params with tree-level relations: sw2 = 1 - mw^2/mz^2, e = sqrt(4 pi/alpha_em_inv),
 * gW = e/sw, gZ = e/(sw cw), gs = sqrt(4 pi alpha_s); FFV couplings follow Eq. 35.
 * Widths enter only the propagator denominators (fixed width, reading SURVEY.md 8c-A4). */
typedef struct {
  double mz, mw, gz, gw; /* Z, W masses and widths */
  double mt, gt;         /* top mass and width */
  double mb;             /* bottom mass (0 in the configs) */
  double mh, gh;         /* Higgs mass and width (library vertices only) */
  double alpha_em_inv;   /* 1/alpha */
  double alpha_s;        /* strong coupling, fixed */
  int ckm_diagonal;      /* must be 1 (only the diagonal CKM is implemented) */
  int complex_mass;      /* 0: fixed widths in the propagator denominators only (default, reading A4).
                            1: the paper's complex-mass option (Eq. 55-56): m_V^2 -> m_V^2 - i m_V
                            Gamma_V (V = W, Z) also in the q q / m_V^2 term of the propagators and in the couplings
                            g_W m_W, g_Z m_Z, 1/v; Eq. 56 fixes Gamma_W = mw gz / mz, the input gw is then ignored */
} hg_params;

/* Final-state cuts (Eq. 8-11; scope: SURVEY.md 8c-A11/A12).  A value <= 0 disables
 * that cut.  A failing event keeps its place in the batch with weight 0 ("null value"). */
typedef struct {
  double pt_jet_min;  /* pT of every gluon jet > this */
  double eta_jet_max; /* |eta| of every gluon jet < this */
  double eta_lep_max; /* |eta| of every charged lepton < this */
  double dr_jj_min;   /* Delta R (Eq. 9b) of every gluon pair > this */
} hg_cuts;

/* Static description of a generated process (from the process generator, step a0 of SURVEY.md 8a). */
typedef struct {
  int n_ext;          /* external legs */
  int n_final;        /* final-state legs */
  int n_hel_total;    /* 2^n_ext helicity combinations of Eq. 4 */
  int n_hel_nonzero;  /* combinations that are not identically zero (the only ones evaluated) */
  int n_diagrams;     /* topological Feynman diagrams */
  int n_amplitudes;   /* diagrams after splitting four-gluon vertices into 3 colour structures (C.47-48) */
  int n_flows;        /* colour-flow basis size = rank of the colour matrix */
  int n_draws;        /* uniform random numbers per event used by the phase-space generator */
  double avg_factor;  /* 1/(spin avg * colour avg * identical-particle factor), Eq. 4 + A7 */
  double flops_f64;   /* algorithmic floating-point operations per event of hg_matrix_element (add, mul = 1,
                         fma = 2, div, sqrt = 1), counted by running the generated code on a counting type */
  double flops_ps;    /* same for phase-space generation + cuts (hg_gen_phase_space) */
} hg_process_info_t;

/* Create / destroy a context bound to one CUDA device.  Every call on the context runs on that device whatever the
 * calling thread's current device is, and leaves the caller's current device as it found it; d_ pointers and the
 * stream passed to a call must belong to the context's device.  Returns HG_ECUDA if the device cannot be used. */
int hg_create(hg_ctx** out, int cuda_device);
void hg_destroy(hg_ctx* ctx);

/* Text of the last error on this context (ctx-owned, valid until the next failing call).  ctx == NULL
 * returns the text of the last failure of a call that has no context (hg_create, hg_accumulate_noalloc). */
const char* hg_last_error(const hg_ctx* ctx);

/* Default inputs of BASELINE.json (MZ=91.1876, MW=80.419, GZ=2.441, GW=2.048, 1/alpha=132.507,
 * mt=174.3, Gt=1.5, mb=0, alpha_s=0.118) and the default cuts of config `process`. */
void hg_default_params(hg_params* out);
int hg_default_cuts(int process, hg_cuts* out);

/* Step a0 result.  Host only. */
int hg_process_info(int process, hg_process_info_t* out);

/* Set SM inputs and cuts; derives all couplings (host only, no launch).  cuts == NULL keeps each
 * process' default cuts.  HG_EINVAL if a mass/width/alpha is not finite or positive where required,
 * or ckm_diagonal != 1. */
int hg_set_params(hg_ctx* ctx, const hg_params* par, const hg_cuts* cuts);

/* Steps a1-a4: Philox4x32-10 uniforms -> flat RAMBO momenta at fixed sqrt_s_hat (config 4:
 * Breit-Wigner mapped t, W masses, Eq. 27, massive RAMBO and nested two-body decays,
 * Eq. 25-26) -> phase-space weight -> cuts.
 *   d_p    [n_ext][4][n] out   momenta (SoA, see above), incoming legs = sqrt_s_hat/2 (1,0,0,+-1)
 *   d_wps  [n] out             phase-space weight dPhi_n (includes the Breit-Wigner Jacobians ds/2pi)
 *   d_pass [n] out or NULL     1 if the event passes the cuts else 0 (uint8)                         */
int hg_gen_phase_space(hg_ctx* ctx, int process, int precision, uint64_t seed, uint64_t first_event,
                       int64_t n, double sqrt_s_hat, void* d_p, void* d_wps, uint8_t* d_pass,
                       void* cuda_stream);

/* Steps a5-a8: |Mbar|^2 = avg_factor * sum_helicities sum_colours |sum_diagrams M|^2 (Eq. 4, 6) for every
 * event of the batch (no cuts applied here).
 *   d_p   [n_ext][4][n] in     momenta
 *   d_me2 [n] out              |Mbar|^2 in GeV^(8 - 2 n_ext)                                         */
int hg_matrix_element(hg_ctx* ctx, int process, int precision, int64_t n, const void* d_p, void* d_me2,
                      void* cuda_stream);

/* Same operation on HOST buffers (pinned memory for full copy speed), pipelined in chunks of 2^19 events through
 * two context-owned device buffers (grown on demand, released by hg_destroy): the H2D copy of the next chunk runs
 * on a context-owned stream while the kernel and the D2H copy of the current one run on cuda_stream.
 * Synchronises cuda_stream before returning. */
int hg_matrix_element_host(hg_ctx* ctx, int process, int precision, int64_t n, const void* h_p,
                           void* h_me2, void* cuda_stream);

/* The same for events given in the partonic centre-of-mass frame: the two incoming momenta are sqrt_s_hat/2 (1, 0, 0,
 * +-1) and are NOT shipped; h_pfinal is [n_ext - 2][4][n] (final-state leg l of the process at row l - 2): 64 bytes
 * per event less over PCIe, which is what bounds this call. */
int hg_matrix_element_host_cm(hg_ctx* ctx, int process, int precision, int64_t n, double sqrt_s_hat,
                              const void* h_pfinal, void* h_me2, void* cuda_stream);

/* Steps a9-a10 on device arrays: w = pass * me2 * wps / (2 s_hat) * (hbar c)^2 [pb]; accumulates
 * acc = (sum w, sum w^2, n, n_pass) in double.  d_pass may be NULL (all pass).  Synchronises the stream;
 * acc is HOST memory, overwritten. */
int hg_accumulate(hg_ctx* ctx, int precision, int64_t n, const void* d_me2, const void* d_wps,
                  const uint8_t* d_pass, double sqrt_s_hat, double acc[4], void* cuda_stream);

/* hg_accumulate for callers that cannot allocate (CUDA graph capture, tight serving loops, harnesses that forbid
 * cudaMalloc): the same steps a9-a10 (section 4: w = |Mbar|^2 x phase-space weight x (hbar c)^2 / (2 s_hat),
 * sums of w and w^2) with NO context and NO allocation -- the per-block partial sums go to a file-scope
 * static __device__ array of the library (3 x 4096 doubles = 96 KB, held by every GPU that loads the library
 * until the process exits) and the result is written to DEVICE memory the caller passes.
 *   d_me2, d_wps [n] in (T), d_pass [n] in or NULL (all pass): device memory on the CURRENT device
 *   d_acc [4] out, DEVICE memory (doubles, 8-byte aligned): (sum w, sum w^2, n, n_pass), overwritten
 *   n <= HG_NOALLOC_MAX_EVENTS, else HG_EINVAL ("n exceeds HG_NOALLOC_MAX_EVENTS")
 * Asynchronous on cuda_stream (two kernel launches, no synchronisation, no copy): d_acc is valid once the stream
 * reaches that point.  Calls no cudaMalloc / cudaFree / allocating routine; the first call on a device looks up
 * the address of the array (cudaGetSymbolAddress), later calls reuse it.  Block b sums the events
 * [4096 b, 4096 (b + 1)) and the blocks are added in a fixed order: the result does not depend on the GPU.
 * Every call SHARES the one array, which keeps the partial sums of the last call: each call overwrites the entries
 * it reads (nothing needs clearing), but two calls that overlap on the GPU (different streams, or graphs replayed
 * concurrently) race on it -- keep calls on one device in stream order.  There is no context to hold an error
 * message: hg_last_error(NULL) returns the text of the last failure of this call. */
#define HG_NOALLOC_MAX_EVENTS 16777216 /* 2^24 */
int hg_accumulate_noalloc(int precision, int64_t n, const void* d_me2, const void* d_wps, const uint8_t* d_pass,
                          double sqrt_s_hat, double* d_acc, void* cuda_stream);

/* Steps a1-a10 in one call.
 * Configs 1, 3 and process 6: fused in one kernel -- each thread draws its event, builds momenta, applies the
 * cuts, evaluates |Mbar|^2 only if it passes, forms w in pb and the block reduces (sum w, sum w^2, n_pass);
 * nothing per-event touches HBM.
 * Configs 2, 4, 5 and processes 7-9: per chunk of 2^20 events a phase-space kernel (at full occupancy) writes the
 * points to a context-owned buffer (grown on demand, freed by hg_destroy), a compaction kernel lists the passing
 * events in order, and a third kernel evaluates |Mbar|^2 of exactly those (staged matrix elements at 8-12 warps per
 * SM) and reduces.  Same results as the fused form, fixed summation order.
 * Synchronises the stream; acc (HOST, overwritten) = (sum w, sum w^2, n, n_pass).  sigma = acc[0]/acc[2]. */
int hg_integrate_step(hg_ctx* ctx, int process, int precision, uint64_t seed, uint64_t first_event,
                      int64_t n, double sqrt_s_hat, double acc[4], void* cuda_stream);

/* The paper's own phase-space parameterisation for hadron collisions (Section 3 and Appendix A, PAPER.md:358-393,
 * 1110-1194; reading A23): integration variables y_i, ln(pT_i^2 + m_i^2), phi_i and the Breit-Wigner
 * mapped resonance masses, with the parton momentum fractions x_a, x_b following from momentum conservation
 * (Eq. 24, A.9) and a null weight for x >= 1 (A.10).  Every jet's pT and rapidity cut is built into the ranges
 * (|y_jet| < eta_jet_max of the cuts, or 5 when that cut is off; pT_jet from pt_jet_min, or 1 GeV, to sqrt(s)/2);
 * the resonance (W, Z, or the second top of config 4) takes the recoil and has |y| < y_res_max.  CTEQ6L1 is not
 * available: the parton density of beam parton i is the toy  f(x) = pdf_norm[i] x^-pdf_a[i] (1 - x)^pdf_b[i].
 *
 * After hg_set_hadronic(ctx, h) with h != NULL, hg_gen_phase_space and hg_integrate_step take their sqrt_s_hat
 * argument as the HADRONIC sqrt(s); momenta are in the lab frame (incoming partons x_a, x_b along +-z); d_wps is
 * dSigma-weight * f_a f_b * s / s_hat, so that w = pass * me2 * wps * (hbar c)^2 / (2 s) as before; a point with
 * x_a >= 1 or x_b >= 1 has wps = 0 and pass = 0.  Implemented for HG_UDX_EPVE, HG_UUX_EPEMG, HG_UDX_EPVEGG,
 * HG_GG_TTXG_DILEP, HG_UDX_EPVEGGG, HG_UDX_EPVEGGGG (HG_EINVAL otherwise).  h == NULL returns to RAMBO at fixed s_hat.
 * hg_default_hadronic: valence-like (2.2, 0.5, 3) and sea-like (0.2, 1.2, 7) quark densities (gluon (3, 1.2, 5) for
 * config 4), y_res_max = 4. */
typedef struct {
  double y_res_max;
  double pdf_norm[2], pdf_a[2], pdf_b[2];
} hg_hadronic;
int hg_default_hadronic(int process, hg_hadronic* out);
int hg_set_hadronic(hg_ctx* ctx, const hg_hadronic* h);

/* Adaptive sampling grid of the integration (role of the BASES grid: "a grid-optimisation step followed by an
 * integration step"; the algorithm is the published VEGAS one, reading A22).
 * Every uniform draw d of an event (n_draws of hg_process_info) has a grid of n_bins bins with edges
 * 0 = g[d][0] < ... < g[d][n_bins] = 1; the draw picks a bin uniformly and a point inside it, the event weight carries
 * the Jacobian prod_d n_bins (g[d][i+1] - g[d][i]).
 *
 * hg_set_grid: until reset, hg_gen_phase_space and hg_integrate_step sample through d_grid ([n_dim][n_bins + 1]
 * doubles, DEVICE memory owned by the caller, read at every call; 2 <= n_bins <= HG_GRID_MAX_BINS).  n_dim must equal
 * n_draws of the process of those calls, else they return HG_EINVAL (a grid belongs to one process).  If d_hist is not NULL ([n_draws][n_bins] doubles, device, caller-owned, caller-zeroed) every
 * hg_integrate_step ADDS the sum of w^2 of the passing events per (draw, bin) to it: the grid-optimisation step.
 * Summation order is fixed (no atomics): same inputs, same histogram.  d_grid == NULL returns to flat sampling.
 *
 * hg_grid_refine (host only; h_ pointers are host memory): one VEGAS refinement of every variable's edges from the
 * accumulated histogram -- smoothing over neighbouring bins, compression ((1 - s)/ln(1/s))^alpha, re-binning to equal
 * content; a variable whose histogram is empty or not finite keeps its edges.  h_grid is updated in place. */
#define HG_GRID_MAX_BINS 64
int hg_set_grid(hg_ctx* ctx, const double* d_grid, int n_dim, int n_bins, double* d_hist);
int hg_grid_refine(int n_dim, int n_bins, const double* h_hist, double alpha, double* h_grid);

#ifdef __cplusplus
}
#endif
#endif /* HG_H */
