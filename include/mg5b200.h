/* mg5b200.h -- C ABI of the B200-native data-parallel matrix-element library.
 *
 * Hot path of arxiv 2507.21039 (CUDACPP plugin of MadGraph5_aMC@NLO): helicity- and colour-summed leading-order
 * tree-level |M|^2 for a batch of phase-space points, plus event-by-event helicity and colour selection.
 * The entry points follow the paper's statement of the interface:
 *   - PAPER.md:152  "Bridge objects can only be constructed, executed, and destroyed"     -> mg_create / mg_compute / mg_destroy
 *   - PAPER.md:481  creation/deletion are expensive and stay out of the event loop           -> long-lived mg_ctx, workspace reuse
 *   - PAPER.md:184, 240  standalone: random numbers -> RAMBO -> matrix elements              -> mg_sample_rambo, mg_sample_uniforms
 *   - PAPER.md:110  only the non-vanishing helicity combinations are summed                 -> mg_filter_helicities
 *   - PAPER.md:132  couplings travel as per-event arrays                                     -> d_gs[nevt]
 *   - PAPER.md:576  precision mode d / f / m chosen up front                                  -> `precision` of mg_create
 *   - PAPER.md:80, 96, 124-128  events adjacent in memory (AOSOA) for coalesced access       -> `layout`
 * Everything the paper leaves open (formulas, RAMBO, Philox addressing, selection rule) follows DESIGN.md.
 *
 * Conventions
 *   - All `d_*` pointers are DEVICE memory owned by the caller, `h_*` pointers are HOST memory owned by the caller.
 *     The library never allocates or frees caller-visible memory; workspace belongs to the context.
 *   - Momenta are FP64 at the boundary in every precision mode, component order (E, px, py, pz), GeV, legs in the
 *     order of the process string (g g -> t t~ g ...: legs 0,1 incoming; e+ e- -> mu+ mu-: e+ e- mu+ mu-).
 *     MG_LAYOUT_AOS:   d_momenta[ievt][ileg][4];
 *     MG_LAYOUT_AOSOA: d_momenta[ievt / 32][ileg][4][ievt % 32]  (nevt must be a multiple of 32).
 *   - Outputs: d_me[nevt] FP64; d_sel_hel[nevt] int32 index into the full 2^npar helicity table
 *     (h = sum_leg b_leg 2^(npar-1-leg), b = (lambda+1)/2); d_sel_col[nevt] int32 index into the colour flows listed
 *     in lexicographic order of gluon leg numbers (0 when ncolor = 1).
 *   - Every function returns 0 on success or a negative MG_E* code; nothing aborts or prints.
 *     mg_strerror() describes a code; after MG_ECUDA it includes the CUDA error string of the failing context call.
 *   - `cuda_stream` is a cudaStream_t passed as void* (NULL = default stream).  mg_compute, mg_sample_* are
 *     asynchronous on that stream; mg_filter_helicities synchronises it (its result is needed on the host).
 *   - Thread safety: one context per host thread.  The calls on one context share its workspace: they may be issued on
 *     different streams, and the library orders them itself (a call on another stream than the previous one first
 *     waits, on the device, for that one), but they never overlap.  Use one context per stream for concurrency.
 */
#ifndef MG5B200_H
#define MG5B200_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct mg_ctx mg_ctx; /* opaque: tables, workspace, good-helicity mask */

/* Standard-Model inputs in GeV (BASELINE.json configs): MZ, WZ, MT, WT, 1/alpha_EW, G_F, alpha_s. */
typedef struct {
  double MZ, WZ, MT, WT, aEWM1, Gf, alpha_s;
} mg_sm_params;

typedef struct {
  int npar;    /* external legs */
  int ndiag;   /* Feynman diagrams (2, 3, 16, 123, 1240) */
  int namp;    /* amplitudes, three colour/Lorentz structures per 4-gluon vertex (2, 3, 18, 159, 1890) */
  int ncolor;  /* colour flows */
  int ncomb;   /* helicity combinations 2^npar */
  int ngood;   /* surviving combinations; -1 before mg_filter_helicities */
  int denom;   /* averaging factor: initial spins x initial colours x identical final-state particles */
  double mass[8];                    /* external masses per leg */
  long long flops_per_event;          /* flops the kernels execute per event (all helicities) */
  long long flops_per_event_canonical;/* flops of the method as the paper runs it (no helicity recycling) */
  int nchannel;/* integration channels of mg_compute_multichannel: diagrams without four-gluon vertices (3, 15, 105, 945); 0 for e+e- */
} mg_info;

enum { MG_EE_MUMU = 1, MG_GG_TT = 2, MG_GG_TTG = 3, MG_GG_TTGG = 4, MG_GG_TTGGG = 5,
       /* Drell-Yan: u(0) u~(1) -> e+(2) e-(3) + 0..3 gluons (legs 4..), photon + Z, all legs massless */
       MG_UU_EE = 6, MG_UU_EEG = 7, MG_UU_EEGG = 8, MG_UU_EEGGG = 9 };
enum { MG_FP64 = 0, MG_FP32 = 1, MG_MIXED = 2, MG_FP32_ALL = 3 };
enum { MG_LAYOUT_AOS = 0, MG_LAYOUT_AOSOA = 1, MG_LAYOUT_SOA = 2 /* host buffers of mg_compute_host only */ };
enum { MG_AOSOA_V = 32 };
enum { MG_OK = 0, MG_EINVAL = -1, MG_ENOTFILTERED = -2, MG_ECUDA = -3, MG_ENOMEM = -4 };

/* Create a context for `process` (MG_EE_MUMU..MG_UU_EEGGG) in `precision` (MG_FP64: everything FP64; MG_FP32:
 * wavefunctions, amplitudes and colour sum in FP32, while the external wavefunctions, gluon-subset momenta and propagator
 * denominators are formed in FP64 from the FP64 momenta and then rounded, helicity sum in FP64; MG_FP32_ALL: those too in
 * FP32 (the paper's FP32 build; reported beside MG_FP32); MG_MIXED: amplitudes FP64,
 * colour-flow amplitudes cast to FP32 for the colour sum) on CUDA device `device`.  Uploads the task program,
 * colour matrix and parameters.  *out receives the context.  Errors: MG_EINVAL (bad argument), MG_ECUDA, MG_ENOMEM. */
int mg_create(mg_ctx** out, int process, const mg_sm_params* sm, int precision, int device);

/* Free the context and its workspace.  NULL is allowed. */
int mg_destroy(mg_ctx* ctx);

/* Process description (host struct filled by the call). */
int mg_get_info(const mg_ctx* ctx, mg_info* out);

/* RAMBO (Kleiss-Stirling-Ellis) flat phase space for `nevt` events with global indices first_event..first_event+nevt-1,
 * driven by Philox4x32-10 uniforms (key = seed, counter = (event, block, purpose 0)); beams along +-z with energy
 * sqrt_s/2 each, final-state masses from the process.  Writes d_momenta in `layout` and, if non-NULL, the phase-space
 * weight d_weight[nevt].  PAPER.md:184.  Errors: MG_EINVAL (NULL, nevt < 0, AOSOA with nevt % 32 != 0), MG_ECUDA. */
int mg_sample_rambo(mg_ctx* ctx, unsigned long long seed, unsigned long long first_event, int nevt, double sqrt_s,
                    int layout, double* d_momenta, double* d_weight, void* cuda_stream);

/* Per-event uniforms in (0,1) for the helicity and colour selection (Philox purpose 1, block 0).  Either output may
 * be NULL. */
int mg_sample_uniforms(mg_ctx* ctx, unsigned long long seed, unsigned long long first_event, int nevt,
                       double* d_rnd_hel, double* d_rnd_col, void* cuda_stream);

/* Helicity filter: evaluates every helicity combination on the given batch and keeps those with
 * |M_h|^2 != 0 (exact compare, rel_threshold = 0) for at least one event; with rel_threshold in (0, 1) the test is
 * |M_h|^2 > rel_threshold * sum_h |M_h|^2 of that event (for processes whose vanishing helicities vanish by
 * cancellation, not term by term).  The mask is cached in the context and used by mg_compute.  *ngood_out
 * (nullable) receives the count, h_good_out (nullable, host, ncomb bytes) the mask.  Synchronises `cuda_stream`.
 * d_gs: per-event strong coupling g_s [nevt] or NULL (= sqrt(4 pi alpha_s)); ignored by MG_EE_MUMU. */
int mg_filter_helicities(mg_ctx* ctx, const double* d_momenta, const double* d_gs, int nevt, int layout,
                         double rel_threshold, int* ngood_out, unsigned char* h_good_out, void* cuda_stream);

/* Install a good-helicity mask (host, ncomb bytes of 0/1, at least one 1) instead of deriving it from a batch: the
 * multi-GPU path ORs the masks of all ranks and installs the union on every rank, so that results do not depend on how
 * the events were split.  Synchronises `cuda_stream`.  Errors: MG_EINVAL. */
int mg_set_good_helicities(mg_ctx* ctx, const unsigned char* h_mask, void* cuda_stream);

/* Matrix elements and selection for one batch: d_me[i] = sum over good helicities of J^dagger C J / denom;
 * d_sel_hel[i] = first good h with r_hel * sum_h |M_h|^2 < running sum; d_sel_col[i] likewise over the colour-flow
 * weights sum_h |J_{h,c}|^2 with r_col.  d_rnd_hel / d_rnd_col / d_sel_hel / d_sel_col may be NULL (selection
 * skipped).  Errors: MG_ENOTFILTERED if mg_filter_helicities has not run, MG_EINVAL, MG_ECUDA, MG_ENOMEM. */
int mg_compute(mg_ctx* ctx, const double* d_momenta, const double* d_gs, const double* d_rnd_hel,
               const double* d_rnd_col, int nevt, int layout, double* d_me, int* d_sel_hel, int* d_sel_col,
               void* cuda_stream);

/* Multichannel single-diagram enhancement (run-card options vector_size and sde_strategy = 1):
 * mg_compute plus, per event, the numerator |A_k|^2 of the event's channel k and the denominator sum_k |A_k|^2, both summed
 * over the good helicities and carrying g_s^(2 ng).  The channels are the Feynman diagrams WITHOUT four-gluon vertices, A_k the
 * colour-stripped value of diagram k; they are numbered from 1 in ascending byte order of their names (a gluon g = 0..ng-1 in
 * process order is one digit, a three-gluon vertex over {A, B}, A holding the lowest label, is "(" A B ")", the blocks along the
 * quark line from t to t~ are joined by "|": g g -> t t~ has channels 1 "(01)", 2 "0|1", 3 "1|0").
 * d_channel[ceil(nevt / 32)]: the channel of every block of MG_AOSOA_V = 32 consecutive events (the paper keeps the channel
 * fixed over a warp-sized block so that the events stay in lockstep); 0 = no channel (numerator 0, colour unrestricted).
 * d_sel_col is selected among the colour flows the channel's diagram contributes to (the last such flow as fall-back).
 * The kernels no longer form one amplitude per diagram for the matrix element, so the channel sums come
 * from a second task program of the same emitter, evaluated in FP64 in every precision mode.
 * d_num[nevt], d_den[nevt]: caller-owned device outputs.  Other arguments, outputs and errors as mg_compute; MG_EINVAL for
 * e+ e- -> mu+ mu- (no channels) and for NULL d_channel / d_num / d_den. */
int mg_compute_multichannel(mg_ctx* ctx, const double* d_momenta, const double* d_gs, const double* d_rnd_hel,
                            const double* d_rnd_col, const int* d_channel, int nevt, int layout, double* d_me,
                            int* d_sel_hel, int* d_sel_col, double* d_num, double* d_den, void* cuda_stream);

/* mg_compute for callers that cannot allocate (CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc):
 * the same kernels and the same results as mg_compute, but the per-helicity and per-flow scratch lives in a static device
 * array of MG_NOALLOC_SCRATCH_BYTES inside the library (every GPU that loads the library holds it until exit) instead of
 * the context's growable workspace.  The call makes no cudaMalloc / cudaFree / allocating library call.
 * Limit: 256 + nevt * 8 * (ncomb + w * ncolor) <= MG_NOALLOC_SCRATCH_BYTES, w = rows of colour-flow partial sums kept per event: 1,
 * except in the FP32 modes of g g -> t t~ g g (2) and g g -> t t~ g g g (4).  In FP64: at most 116506 / 55187 / 23830 / 8456 events per
 * call for g g -> t t~ / t t~ g / t t~ g g / t t~ g g g, 123360 for e+ e- -> mu+ mu-; a larger nevt is rejected with MG_EINVAL and a
 * message that states the limit for the context at hand.
 * All calls, of every context on a device, share the one array; it keeps the previous call's contents (what must start
 * from zero is cleared on the stream by the call itself).  Calls that overlap on the GPU -- two contexts, or one context
 * driven from two host threads -- therefore race: order them on one stream or with events.  Calls on ONE context are
 * ordered by the library as for mg_compute.  mg_get_last_details does not see a batch computed through this entry point.
 * Arguments, outputs and the other errors are those of mg_compute (the helicity mask must be installed beforehand). */
enum { MG_NOALLOC_SCRATCH_BYTES = 16 << 20 };
int mg_compute_noalloc(mg_ctx* ctx, const double* d_momenta, const double* d_gs, const double* d_rnd_hel,
                       const double* d_rnd_col, int nevt, int layout, double* d_me, int* d_sel_hel, int* d_sel_col,
                       void* cuda_stream);

/* Host bridge ("Bridge ... handles internal memory management (such as transposition between column- and
 * row-major layout)"; once the matrix element is fast the host side limits event generation): the same
 * as mg_compute with HOST buffers (pinned memory recommended; pageable memory works but its copies do not overlap).
 * The batch is cut into about 8 chunks of whole 32-event pages (at least 8192 events each) that run through two internal
 * lanes -- stream, staging buffers and workspace each -- so that the H2D copy of one chunk, the kernels of another and the
 * D2H copy of a third overlap; one cudaMemcpyAsync per buffer per chunk.  The lanes start after the work queued on
 * `cuda_stream` and the call returns when all results are on the host.  Results are bit-identical to mg_compute's.
 * `layout` describes h_momenta: MG_LAYOUT_AOS, MG_LAYOUT_AOSOA, or MG_LAYOUT_SOA = h_momenta[c][ileg][ievt] (ievt fastest: the
 * column-major image of [nevt][npar][4], a Fortran array P(NEVT, NPAR, 0:3)), which is transposed on the device.
 * h_gs, h_rnd_*, h_sel_* may be NULL as in mg_compute. */
int mg_compute_host(mg_ctx* ctx, const double* h_momenta, const double* h_gs, const double* h_rnd_hel,
                    const double* h_rnd_col, int nevt, int layout, double* h_me, int* h_sel_hel, int* h_sel_col,
                    void* cuda_stream);

/* Diagnostics of the last mg_compute / mg_filter_helicities batch, resident in the context's workspace:
 * per-helicity |M_h|^2 (d_mh2[nevt][ncomb]) and colour-flow weights (d_wcol[nevt][ncolor]) copied to caller-owned
 * device buffers (either may be NULL).  Used by the parity tests. */
int mg_get_last_details(mg_ctx* ctx, int nevt, double* d_mh2, double* d_wcol, void* cuda_stream);

/* Register-only FMA-chain microbenchmark: returns the sustained FMA rate of the plain FP64
 * (precision MG_FP64) or FP32 (MG_FP32) pipe in TFLOP/s in *tflops_out; `millis` is the target run length. */
int mg_measure_fma_peak(mg_ctx* ctx, int precision, double millis, double* tflops_out);

/* FP64 pipe microbenchmarks for the colour-sum decision (the colour sum as one
 * matrix multiplication): one 512-thread CTA per SM runs mode 0 DFMA register chains, 1 DMMA (mma.sync m8n8k4 f64)
 * register chains, 2 both interleaved in every warp, 3 both on alternating warps, 4 DMMA fed from shared memory in the
 * layout of the colour-flow amplitude tile (64 rows x K = 120, matrix fragments), 5 the DFMA colour form fed from
 * shared memory.  out[0] = plain-FMA TFLOP/s, out[1] = tensor TFLOP/s achieved in that mode, out[2] = milliseconds per
 * iteration of the benchmark body.  `millis` is the target run length. */
int mg_measure_fp64_pipes(mg_ctx* ctx, int mode, double millis, double* out);

/* Number of kernel launches issued by this context since creation (for bench.py's gpu_launches). */
long long mg_launch_count(const mg_ctx* ctx);

/* Device timing of the dominant kernel (the amplitude kernel that mg_compute / mg_filter_helicities launch): when
 * enabled, the library records a CUDA event pair around that launch on the caller's stream.  mg_kernel_time_ms waits
 * for the recorded launches, returns their summed duration and count, and clears the record.  Used by bench.py for
 * the roofline figure; off by default. */
int mg_enable_kernel_timing(mg_ctx* ctx, int on);
int mg_kernel_time_ms(mg_ctx* ctx, double* total_ms, long long* nlaunch);

const char* mg_strerror(int code);

#ifdef __cplusplus
}
#endif
#endif /* MG5B200_H */
