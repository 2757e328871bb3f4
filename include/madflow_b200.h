/* madflow_b200.h -- C-ABI boundary of the B200-native MadFlow leading-order integrand path.
 *
 * The operation: "integrate an event-parallel integrand with an adaptive importance-sampling
 * integrator, entirely on the device" (PAPER.md:15 parallelism over events; PAPER.md:29 the four
 * ingredients: integrator, PDF interpolation, phase space + cuts, matrix element
 * VegasFlow/PDFFlow; PAPER.md:59 pipeline "random numbers -> phase-space kinematics -> matrix
 * element -> histogram accumulation"; PAPER.md:85 everything stays in GPU memory).  The paper prints
 * no formulas; the arithmetic of every step is the reading listed in DESIGN.md (O1-O11, A1-A24).
 *
 * Conventions
 *  - Every function returns MF_OK (0) or a negative MF_E* code; none throws or exits.  A message for
 *    the last error of the calling thread is available from mf_last_error().
 *  - mf_vegas_t is opaque and owned by the library (create/destroy).  The library owns its scratch
 *    (per-block partial sums, grid edges, iteration records) in device memory.
 *  - Pointers in mf_config_t and the "host_*" arguments are HOST pointers.  Pointers inside
 *    mf_eval_out_t are DEVICE pointers owned by the caller (e.g. torch tensors' data_ptr()).
 *  - `cuda_stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).  Work is
 *    only enqueued; a call synchronises the stream only where stated.
 *  - Event indices are global within an iteration: evaluating [0,N) in one call or in chunks gives
 *    identical per-event values (counter-based RNG, reading A1).
 *  - There is no CPU fallback: without a CUDA device every compute call returns MF_ECUDA.
 */
#ifndef MADFLOW_B200_H
#define MADFLOW_B200_H
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef struct mf_vegas mf_vegas_t;

enum { MF_OK = 0, MF_EINVAL = -1, MF_ENOMEM = -2, MF_ECUDA = -3, MF_ESTATE = -4, MF_EUNSUPPORTED = -5 };
/* processes (BASELINE.json configs 0-3; 4 = the quark channel of SURVEY 8(f)2) */
enum { MF_EE_MUMU = 0, MF_GG_TT = 1, MF_GG_TTG = 2, MF_GG_TTGG = 3,
       MF_QQ_TT = 4, MF_PP_TT = 5, MF_QQ_TTG = 6, MF_QG_TTQ = 7 };
                           /* MF_QQ_TT: quark channel ("any process generated (at LO)"): q q~ -> t t~, one
                            * s-channel-gluon diagram, averaged over 4 helicities x 9 colours, with the parton luminosity
                            * summed over the five light flavours and both beam orientations:
                            *   F = J_V J_x [sum_q f_q(x1) f_q~(x2) + f_q~(x1) f_q(x2)] |M|^2 W_PS K / (2 shat).
                            * Kinematics, VEGAS dimensions and selectable generators of process 1; fused path.  Needs the
                            * 11-flavour grid (pdf_nf = 11).  mf_eval_out_t.pdf then holds the two flavour sums
                            * sum_q xf_q(x1) xf_q~(x2) and sum_q xf_q~(x1) xf_q(x2).
                            * MF_PP_TT = 5: p p -> t t~ at LO, the subprocesses g g -> t t~ and q q~ -> t t~ in one integrand,
                            *   F = J_V J_x [xg(x1) xg(x2) |M_gg|^2 + (L12 + L21) |M_qq|^2] / (x1 x2) W_PS K / (2 shat)
                            * on the same grid (gluon = table 5); mf_eval_out_t.pdf = {xg(x1) xg(x2), L12 + L21}, me2 = the
                            * luminosity-weighted mean of the two |M|^2.
                            * MF_QQ_TTG = 6, MF_QG_TTQ = 7 (SURVEY 8(f)2 "q q~ -> t t~ (g), q g -> t t~ q"): the channels with a
                            * second quark line and one gluon, five diagrams each; kinematics, VEGAS dimensions (7, or 14), cuts
                            * (ptmin_g, etamax_g on the third final particle: the gluon, resp. the light-quark jet) and selectable
                            * generators of process 2; 11-flavour grid; fused path.
                            *   6: F = J_V J_x [L12 |M(q(p1) q~(p2) -> t t~ g)|^2 + L21 |M(q~(p1) q(p2) -> t t~ g)|^2] / (x1 x2) W_PS K / (2 shat)
                            *      (the two |M|^2 differ: charge asymmetry); pdf = {L12, L21}, me2 = their weighted mean |M|^2.
                            *   7: the four channels q g, g q, q~ g, g q~ -> t t~ + q/q~ with Lqg = sum_q xf_q(x1) xg(x2) etc.;
                            *      pdf = {Lqg + Lq~g, Lgq + Lgq~}, me2 = the luminosity-weighted mean of the four |M|^2.          */

/* Selectable generators (the paper fixes no phase-space algorithm):
 *  MF_GEN_CLASSIC_RAMBO  textbook RAMBO (Kleiss, Stirling, Ellis 1986) from 4 n_final uniforms in place of the
 *                        3 n_final - 4-random sequential form (reading O4), then the same massive rescaling;
 *                        VEGAS dimensions d = 2 + 4 n_final (10, 14, 18).
 *  MF_GEN_LINEAR_TAU     tau = tau0 + (1 - tau0) y0 in place of tau = tau0^(1-y0) (reading O3);
 *                        J_x = (1 - tau0)(-ln tau).
 * Both sample the same integral: the cross section agrees with the default generators' within errors.
 * Processes 2 and 3 run them on the staged path only (mf_set_path(h, 0) -> MF_EUNSUPPORTED). */
enum { MF_GEN_CLASSIC_RAMBO = 1, MF_GEN_LINEAR_TAU = 2 };

typedef struct {
  uint32_t struct_size;      /* = sizeof(mf_config_t); ABI check                                     */
  int32_t  process;          /* MF_EE_MUMU .. MF_QG_TTQ                                              */
  int32_t  precision;        /* 64 (fp64, the path); 32 = mixed precision, process MF_GG_TTG only: |M|^2
                              * (S7) in fp32, everything else (S1-S6, S8-S10) in fp64; staged path and
                              * mf_integrand_eval; other processes -> MF_EUNSUPPORTED                  */
  int32_t  device;           /* CUDA ordinal                                                         */
  uint64_t seed;             /* Philox key (reading A1)                                              */
  uint32_t n_bins;           /* VEGAS bins per dimension, 1..64 (configs: 50)                        */
  uint32_t generator;        /* MF_GEN_* flags, processes 1-3; 0 = the generators of the configs */
  double   alpha_damp;       /* VEGAS damping exponent (1.5)                                         */
  double   sqrt_s;           /* collider energy, GeV (config 0: the fixed e+e- energy)               */
  double   m_top, alpha_s, alpha_em, mu_f;
  double   ptmin_g, etamax_g, drmin_gg;   /* cuts on final gluons, lab frame; <= 0 disables (O7)     */
  double   gev2_to_pb;       /* 0.3894e9 (reading A11)                                               */
  const double *pdf_xf;      /* HOST [pdf_nx][pdf_nq] row-major table of x*g(x,Q^2); copied at       */
                             /* create; required for processes 1-3, ignored for process 0            */
  uint32_t pdf_nx, pdf_nq;   /* knots, uniform in ln x resp. ln Q^2; nx*nq*8 bytes <= 160 KB         */
  double   pdf_xmin, pdf_xmax, pdf_qmin, pdf_qmax;
  uint32_t pdf_nf;           /* flavour tables in pdf_xf: 0 or 1 = the gluon table [nx][nq] (processes 1-3);         */
  uint32_t reserved1;        /* 11 = [11][nx][nq], flavour index = PDG id + 5 (b~ c~ s~ u~ d~ g d u s c b): processes 4-7.  */
                             /* The library stages the tables flavour-innermost in shared memory, keeping             */
                             /* the <= 4 Q^2 rows the stencil of the fixed mu_f touches (36 KB)                     */
} mf_config_t;

/* Optional per-event outputs of mf_integrand_eval.  DEVICE pointers, caller-owned, NULL = skip.     */
typedef struct {
  double  *weight;           /* [n]  F_i = w_i f_i (= t_i * N), pb; 0 for events failing the cuts    */
  double  *x;                /* [n][d]  VEGAS points y_j (O2)                                         */
  uint8_t *bins;             /* [n][d]  VEGAS bin indices k_j                                         */
  double  *momenta;          /* [n][2+n_final][4]  (E,px,py,pz), partonic CM frame, incoming first   */
  double  *me2;              /* [n]  |M|^2 averaged/summed, before the symmetry factor; 0 if cut     */
  double  *pdf;              /* [n][2]  xg(x1,muF^2), xg(x2,muF^2); process 4: the two flavour sums L12, L21;     */
                             /*         process 5: xg(x1) xg(x2) and L12 + L21 (see MF_QQ_TT / MF_PP_TT above) */
  uint8_t *pass;             /* [n]  1 if the event passed the cuts (always 1 for processes 0, 1, 4, 5: no cuts) */
} mf_eval_out_t;

typedef struct { double integral, sigma; uint64_t n_events, n_pass, n_nonfinite; float kernel_ms; } mf_iter_t;
typedef struct { double integral, sigma, chi2_dof; uint32_t n_iter; } mf_result_t;

/* Validate cfg, copy it and the PDF table, allocate device state, set the uniform grid.  No kernel
 * work.  Errors: MF_EINVAL (bad field, kinematics outside the PDF grid), MF_EUNSUPPORTED
 * (precision other than 64, or 32 for a process other than MF_GG_TTG), MF_ECUDA (no device /
 * allocation failure).  Every call leaves the caller's current CUDA device as it found it.           */
int mf_vegas_create(const mf_config_t *cfg, mf_vegas_t **out);
int mf_vegas_destroy(mf_vegas_t *h);
/* d = VEGAS dimensions (2 for process 0, else 2 + 3 n_final - 4, or 2 + 4 n_final with MF_GEN_CLASSIC_RAMBO),
 * n_final = final-state particles */
int mf_ndim(const mf_vegas_t *h, uint32_t *d, uint32_t *n_final);

/* S1-S8 for events [first_event, first_event + n_events) of iteration `iteration` on the CURRENT
 * grid; writes the requested per-event records.  No grid update, no reduction, no host sync.       */
int mf_integrand_eval(mf_vegas_t *h, uint32_t iteration, uint64_t first_event, uint64_t n_events,
                      const mf_eval_out_t *out, void *cuda_stream);

/* One VEGAS iteration of n_events (>= 2) events (random numbers -> phase space -> matrix
 * element -> accumulation), then S10 in a one-block finalize kernel: I, sigma, grid refinement, record
 * appended on the device.  S1-S9 run either FUSED in one kernel (no per-event global traffic; the only
 * path of processes 0 and 1) or STAGED (default for processes 2 and 3, mf_set_path): front end,
 * |M|^2 and reductions as three kernels, each at its own occupancy, with 4 n_final + 3 doubles per
 * cut-passing event passed through a library-owned device workspace (grown on demand, at most 2^24
 * events per launch; larger iterations are processed in slices).  Enqueue only, unless
 * host_out_or_null != NULL: then the stream is synchronised and the iteration record (kernel_ms =
 * device time of the dominant kernel: fused kernel or |M|^2 stage) is returned.                      */
int mf_vegas_iterate(mf_vegas_t *h, uint64_t n_events, void *cuda_stream, mf_iter_t *host_out_or_null);

/* Sharded form of one iteration (multi-GPU): accumulate events
 * [first_event, first_event+n_events) of an iteration of n_total events into the handle's raw sums
 * (device, [2 + d*n_bins] doubles + 2 counters); read / overwrite the raw sums from the host (the
 * caller all-reduces them); finish the iteration from the raw sums.  mf_vegas_iterate ==
 * accumulate(0, n, n) + finalize.                                                                   */
int mf_vegas_accumulate(mf_vegas_t *h, uint64_t first_event, uint64_t n_events, uint64_t n_total,
                        void *cuda_stream);
int mf_get_accum(mf_vegas_t *h, double *host_acc /* [mf_accum_len()] = [2 + d*n_bins] without observables */, uint64_t *host_counts /* [2] */);
int mf_set_accum(mf_vegas_t *h, const double *host_acc, const uint64_t *host_counts);
int mf_vegas_finalize(mf_vegas_t *h, uint64_t n_total, void *cuda_stream, mf_iter_t *host_out_or_null);
/* The same exchange without host round trips (enqueue only, no synchronisation): clear the raw sums; copy them, followed
 * by the two counters converted to double (exact below 2^53), into / from a caller-owned DEVICE buffer of
 * mf_accum_len() + 2 doubles -- one buffer for one all-reduce (e.g. ncclAllReduce / torch.distributed on the same stream). */
int mf_zero_accum(mf_vegas_t *h, void *cuda_stream);
int mf_get_accum_device(mf_vegas_t *h, double *dev_out, void *cuda_stream);
int mf_set_accum_device(mf_vegas_t *h, const double *dev_in, void *cuda_stream);

/* Observable histograms filled in the same pass as the integral ("histogram accumulation";
 * dsigma/dpT of the top quark is the paper's physics plot).  For every event with weight
 * F_i != 0, t_i = F_i / N: sum[o][b] += t_i, sum2[o][b] += t_i^2 with b = floor((v-lo)/(hi-lo)*n_bins)
 * for lo <= v < hi, slot 62 for v < lo (underflow), slot 63 for v >= hi (overflow); v from the final-state
 * momenta (partonic CM frame; all kinds are invariant under the boost along the beam).  At most
 * MF_MAX_OBS observables of at most 62 bins; each histogram has MF_OBS_SLOTS = 64 slots.
 * mf_set_observables copies the definitions and clears the accumulated histograms (n_obs = 0 turns the
 * feature off).  Every finalized iteration adds its histograms to the accumulated ones;
 * mf_get_observables returns them ([n_obs][64] doubles each, host) and the number of iterations summed
 * (divide by it, and by the bin width, for dsigma/dv).  While observables are set, the raw-sum vector
 * of the sharded form (mf_get_accum / mf_set_accum) has mf_accum_len() = 2 + d*n_bins + 2*MF_MAX_OBS*64
 * entries (this iteration's observable sums behind the VEGAS sums).  Processes 2 and 3 fill them on the
 * staged path only (MF_EUNSUPPORTED from mf_vegas_accumulate on the fused path).                     */
enum { MF_OBS_PT_1 = 0, MF_OBS_PT_2 = 1, MF_OBS_M_12 = 2, MF_OBS_PT_3 = 3 };
#define MF_MAX_OBS 4
#define MF_OBS_SLOTS 64
typedef struct { int32_t kind; uint32_t n_bins; double lo, hi; } mf_observable_t;
int mf_set_observables(mf_vegas_t *h, const mf_observable_t *obs, uint32_t n_obs);
int mf_get_observables(mf_vegas_t *h, double *host_sum, double *host_sum2, uint32_t *n_iter);
int mf_accum_len(const mf_vegas_t *h, uint32_t *n);

/* O11 combination over all iterations so far, enqueued behind the last call that changed the integrator
 * state, on that call's stream, which is then synchronised.  MF_ESTATE if no iteration has been run.
 * Stream ordering in general: calls may be issued on different streams; a call that reads or writes the
 * integrator state (grid, raw sums, records) waits on the device for the last call that wrote it, a call
 * that writes the grid also for evaluations in flight; host reads (get_*, result) wait for both.        */
int mf_result(mf_vegas_t *h, mf_result_t *host_out);
/* Checkpoint / resume of the integrator state (an auxiliary of the path: the integration state lives on the device):
 * the grid edges, the per-iteration records, the iteration counter (= the Philox counter word of the next iteration) and the
 * accumulated observable histograms, as one opaque host blob of mf_state_size() bytes (it grows by 40 bytes per iteration).
 * mf_get_state waits for the work in flight and copies it out; mf_set_state puts a blob into a handle created with the SAME
 * configuration (process, generator, dimensions, bins, seed: MF_EINVAL otherwise; observables must have been set as when it was saved):
 * the next mf_vegas_iterate then continues the run bit for bit, and mf_result combines the restored iterations with the new ones. */
int mf_state_size(const mf_vegas_t *h, uint64_t *bytes);
int mf_get_state(mf_vegas_t *h, void *host_buf, uint64_t bytes /* >= mf_state_size */);
int mf_set_state(mf_vegas_t *h, const void *host_buf, uint64_t bytes);
/* per-iteration records; host_out[n_iter] must hold at least max_iter entries; *n_iter = stored    */
int mf_get_iterations(mf_vegas_t *h, mf_iter_t *host_out, uint32_t max_iter, uint32_t *n_iter);
int mf_get_grid(mf_vegas_t *h, double *host_edges /* [d][n_bins+1] */);
int mf_set_grid(mf_vegas_t *h, const double *host_edges);   /* edges must start at 0, end at 1, increase */
/* Launch geometry of the fused kernel: blocks per SM (0 = library default) and threads per block
 * (0 = default).  Results are deterministic for a fixed geometry.                                  */
int mf_set_launch(mf_vegas_t *h, uint32_t blocks_per_sm, uint32_t threads_per_block);
/* Select the iteration path: staged != 0 -> staged (MF_EUNSUPPORTED for processes 0 and 1, which
 * only have the fused kernel), 0 -> fused.  Both give the same per-event values; the summation
 * order (hence the last bits of the sums) differs.                                                   */
int mf_set_path(mf_vegas_t *h, int32_t staged);
/* Device times of the three stages (front end, |M|^2, reductions; ms3[3], host) of the last staged
 * launch (the last SLICE of an iteration of more than 2^24 events: use mf_stage_ms_sum for the whole).
 * MF_ESTATE if the last accumulate ran the fused path.  Waits for the events.                       */
int mf_last_stage_ms(const mf_vegas_t *h, float *ms3);
/* Sums of the three stage times over ALL staged launches (every slice of every iteration) since the
 * previous call, and their number (*launches; at most the last 256 are kept); resets the count.  The
 * events are recorded on the caller's stream inside mf_vegas_accumulate, nothing synchronises until this
 * call, which waits for the last of them.                                                            */
int mf_stage_ms_sum(mf_vegas_t *h, float *ms3, uint32_t *launches);
/* Device times (CUDA events on the caller's stream): of the dominant S1-S9 kernel (fused kernel, or
 * the |M|^2 stage of the staged path) of the last
 * mf_vegas_accumulate / mf_vegas_iterate, and of the whole last mf_vegas_iterate (memsets + fused
 * kernel + reduce + finalize).  Waits for those events to complete.                                 */
int mf_last_kernel_ms(const mf_vegas_t *h, float *fused_kernel_ms, float *iteration_ms);
/* Exact add/mul/fma counts per event of the generated |M|^2 code of the handle's process on the handle's CURRENT path
 * (generator-counted: loop invariants counted once): flops = add + mul + 2 fma.  gg -> tt~g:
 * 11 591 on the staged fp64 path (helicity loop over one gluon), 15 023 on the fused path, in mf_integrand_eval and with the
 * fp32 |M|^2 stage (loop over two gluons: the register-resident organisation).                          */
int mf_me_flops(const mf_vegas_t *h, uint64_t *n_add, uint64_t *n_mul, uint64_t *n_fma);
/* flops per event of the LEANEST organisation of the same amplitude the build-time generator knows (every helicity
 * configuration unrolled, every subexpression shared: gg -> tt~g 11 302, gg -> tt~gg 170 880; other processes: the count
 * of mf_me_flops), and the flops the kernels EXECUTE per event for S7 (= mf_me_flops, except gg -> tt~gg: four lanes per
 * event, each with its own prologue and a share of recomputation).  mf_me_flops lies between the two.        */
int mf_me_flops_bounds(const mf_vegas_t *h, uint64_t *flops_min, uint64_t *flops_executed);
/* S9 (reading O9) as ONE entry point that ALLOCATES NOTHING -- no cudaMalloc, cudaFree or allocating library routine at
 * any call, the first included -- for callers that cannot allocate (code under CUDA graph capture, tight serving loops,
 * harnesses that forbid it).  From n_events per-event weights F_i (dev_weight[n], as mf_integrand_eval writes them) and
 * their VEGAS bins (dev_bins[n][d], uint8) it writes, or with accumulate != 0 adds, into the caller's DEVICE buffer
 * dev_acc[2 + d*n_bins]:  sum_i t_i,  sum_i t_i^2,  H[j][k] = sum_{i in bin k of dimension j} t_i^2,  t_i = F_i / n_total
 * -- the raw-sum vector of mf_vegas_accumulate / mf_set_accum_device (non-finite weights count as 0; fixed summation
 * order for a given n_events).  It is a variant of the library's reduction stage whose scratch (one partial record per
 * CTA) is a file-scope static __device__ array of 296 x (2 + 18 x 64) doubles = 2.7 MB that every GPU loading the library
 * holds until exit.  Limits: d <= 18, n_bins <= 64 (MF_EINVAL beyond; n_events is not limited).  `device` = the CUDA
 * ordinal the buffers live on.  Enqueue only; no synchronisation.  Every call shares the scratch array: calls that
 * overlap on the GPU (different streams without ordering, several host threads) RACE on it -- issue them on one stream
 * or order them with events.  Together with mf_integrand_eval, mf_set_accum_device and mf_vegas_finalize (none of
 * which allocates) a whole iteration of any process runs without the on-demand workspace of mf_vegas_accumulate.      */
int mf_reduce_weights_noalloc(int32_t device, const double *dev_weight, const uint8_t *dev_bins, uint64_t n_events,
                              uint32_t d, uint32_t n_bins, double n_total, int32_t accumulate, double *dev_acc,
                              void *cuda_stream);
/* Register-resident DFMA-chain microbenchmark on `device`: measured fp64 FLOP/s (roofline peak).   */
int mf_fp64_peak(int32_t device, double seconds, double *host_flops_per_s);
const char *mf_last_error(void);

#ifdef __cplusplus
}
#endif
#endif
