/*
 * gbfit.h -- C ABI of the B200-native Galactic-binary (GB) waveform + delta-log-likelihood hot path
 *            of the "Erebor" LISA global fit (arxiv 2405.04690; citations are PAPER.md:<line>).
 *
 * What the library computes
 *   gb_waveform         frequency-domain TDI A/E waveform of each GB on its own N-bin window around f0,
 *                       by the fast/slow decomposition (sec. II.A; App. F):
 *                       the slow LISA response at N time samples (TDI generation 1.5, equal constant arms,
 *                       PAPER.md:105; A,E of Eq. 6) followed by a length-N FFT.
 *   gb_delta_loglike    the change of the Gaussian log-likelihood (Eq. 1-2) when one source
 *                       is added (Eq. 4), removed, or swapped for another (Eq. 5,
 *                       PAPER.md:96-103), against the walker's residual r = d - H and that walker's PSD;
 *                       sums run only over the bins where the source lives.
 *   gb_residual_update  the residual refresh of Algorithm 1: accepted waveforms are
 *                       scatter-added into the per-walker residuals.
 * The paper does not print the GB waveform equations; the exact definition implemented is
 * written out in DESIGN.md ("The path", steps O1-O9) together with every reading of a silent point.
 *
 * General conventions
 *   - Every pointer is a DEVICE pointer on the context's device unless the parameter comment says HOST.
 *     The caller owns every buffer; the library allocates only inside gb_ctx (tables and scratch).
 *   - All calls return an int status (GB_OK = 0, negative = error), never throw, never abort.
 *   - Device work is enqueued on `stream` (a cudaStream_t passed as void*; NULL = the legacy default
 *     stream) and is asynchronous with respect to the host, except the *_host entry points, which
 *     synchronise `stream` before returning (also on every error return: no copy from or into a caller's
 *     host buffer is in flight once a *_host call has returned).  Errors detectable at launch are returned at
 *     once; per-row errors set bits of a sticky device flag that the next call to gb_check() reports:
 *       1  walker index / PSD row out of range, N not in {128,256,512,1024} (gb_waveform: N_b > Nmax), bad move,
 *          or a per-row move whose parameter array is NULL: the row is NOT computed, its dlnL is NaN (waveform
 *          rows are left untouched, update rows are not applied);
 *       2  the window extends beyond the Nyquist bin Tobs / (2 dt): the row IS computed and its output is finite
 *          (the waveform definition does not depend on dt, reading S10) -- the flag is a warning;
 *       4  gb_delta_loglike_keep: sum_n_bins too small: dlnL of every row is still computed and finite, windows
 *          past the capacity are not kept, and gb_residual_update_kept skips (and flags) exactly those rows;
 *          gb_delta_loglike_accept: store_bins too small: rows that no longer fit are reported rejected.
 *   - Complex arrays are complex128, interleaved (re, im) doubles.  Real arrays are f64.
 *   - params row (8 f64): [amp, f0 (Hz), fdot (Hz/s), phi0, cos(iota), psi, lambda (ecl. lon.), sin(beta)].
 *   - Frequency bins: global bin k  <->  f = k / Tobs  (the rfft grid of the data).
 *     A source's window is bins kmin .. kmin+N-1 with kmin = floor(f0*Tobs + 0.5) - N/2.
 *   - Residual semantic r = d - H: ADD subtracts the waveform, REMOVE adds it, SWAP adds old, subtracts new.
 *   - Window bins outside the stored band [k_lo, k_lo + n_f) contribute nothing to any inner product and
 *     are not scattered.
 *   - gb_waveform / gb_delta_loglike / gb_residual_update apply no tempering, prior or proposal density (Eq. 13,
 *     PAPER.md:197): the caller does accept/reject.  gb_delta_loglike_accept, gb_band_sweep(_generate) and gb_temper_sweep
 *     take the decision themselves (inverse temperatures, log q and the uniform draws are inputs, or generated in the
 *     kernel).  Rows of one batched call are evaluated independently against the same residual snapshot.
 *   - A gb_ctx may be used from one host thread at a time.
 */
#ifndef GBFIT_H
#define GBFIT_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct gb_ctx gb_ctx; /* opaque; owns orbit tables, FFT twiddles and scratch on one device */

typedef struct {      /* HOST POD, copied by gb_create */
    double Tobs;      /* observation time [s]; the FFT grid is k / Tobs                 (31457280)           */
    double dt;        /* cadence of the data [s]; only used to validate kmin+N-1 <= Tobs/(2 dt)   (5)         */
    double armlength; /* L [m]                                                          (2.5e9)              */
    double au;        /* astronomical unit [m]                                          (1.495978707e11)     */
    double year;      /* orbital period of the constellation [s]                        (31558149.763545603) */
    double kappa;     /* initial orbital phase of the guiding centre [rad]              (0)                  */
    double lambda0;   /* initial orientation of the constellation [rad]                 (0)                  */
    int32_t device;   /* CUDA device ordinal                                                                 */
    int32_t reserved; /* set to 0                                                                            */
} gb_config;

typedef struct {      /* HOST POD describing DEVICE-resident data, caller-owned */
    double *resid;              /* [n_walkers][2][n_f] complex128; ch 0 = A, ch 1 = E; r = d - H; 16-byte aligned */
    const double *psd;          /* [n_psd][2][n_f] f64; S_n(f) per channel, or 1/S_n if psd_is_inverse           */
    const int32_t *walker_psd;  /* [n_walkers] -> psd row; NULL = identity, or row 0 when n_psd == 1             */
    int64_t k_lo, n_f;          /* residual element i  <->  global bin k_lo + i                                  */
    int32_t n_walkers, n_psd, psd_is_inverse, reserved;
} gb_data;

enum { GB_ADD = 0, GB_REMOVE = 1, GB_SWAP = 2 };

enum {
    GB_OK = 0,
    GB_ERR_INVALID = -1,   /* NULL required pointer, B < 0, bad N, bad config                    */
    GB_ERR_CUDA = -2,      /* a CUDA runtime call failed; see gb_last_error                      */
    GB_ERR_NOMEM = -3,     /* scratch allocation failed                                          */
    GB_ERR_ROW = -4        /* gb_check: row-error flag bits 1 / 2 / 4 of an earlier call (see above) */
};

/* Fill *cfg with the defaults listed above (device 0).  cfg: HOST. */
void gb_default_config(gb_config *cfg);

/* Create a context on cfg->device: builds the orbit tables (analytic equal-arm orbits, O2) for
 * N = 128, 256, 512, 1024 and the FFT twiddles.  cfg, out: HOST.  Returns GB_OK or an error. */
int gb_create(const gb_config *cfg, gb_ctx **out);

/* Free the context and its device memory (synchronises the device).  NULL is allowed. */
void gb_destroy(gb_ctx *ctx);

/* Last error message of this context (HOST string owned by ctx, valid until the next call). */
const char *gb_last_error(const gb_ctx *ctx);

/* Synchronise `stream`, then report and clear the sticky per-row error flag: GB_OK, GB_ERR_ROW or GB_ERR_CUDA. */
int gb_check(gb_ctx *ctx, void *stream);

/* Library version string "gbfit-b200 x.y" (HOST, static). */
const char *gb_version(void);

/* Number of kernels launched by this context since creation (bench.py's gpu_launches counter). */
int64_t gb_launch_count(const gb_ctx *ctx);

/* Bytes of device scratch the context holds right now (work lists, source records, window stores, caches, staging of the
 * *_host forms; grown on demand by the calls, freed by gb_destroy).  Tables (orbit, twiddles) are not counted. */
int64_t gb_scratch_bytes(const gb_ctx *ctx);

/*
 * gb_measure_fp64_peak -- diagnostic, not on the hot path: times a register-only stream of independent DFMAs
 * (8 chains per thread, 512 threads per SM, every SM) on the context's device and returns the sustained rate.
 * This is the measured denominator of the "alu" roofline bench.py reports beside the nominal
 * 148 SMs x 64 DFMA/clk x 2 x clock figure (the delta-lnL path is bound by the plain FP64 pipe).
 *   tflops_out            HOST, 2 flop per DFMA
 *   dfma_per_clk_sm_out   HOST, DFMA lanes per SM per clock at clock_mhz (may be NULL)
 *   clock_mhz             SM clock to normalise by (e.g. the max SM clock); ignored if dfma_per_clk_sm_out is NULL
 * Synchronises `stream`.  Returns GB_OK or GB_ERR_INVALID / GB_ERR_CUDA.
 */
int gb_measure_fp64_peak(gb_ctx *ctx, double *tflops_out, double *dfma_per_clk_sm_out, double clock_mhz, void *stream);

/*
 * gb_waveform -- A/E windows of B sources.
 *   params   [B][8] f64
 *   N        window length used for every row when n_bins == NULL; one of 128, 256, 512, 1024
 *   n_bins   [B] int32 per-row window length, or NULL
 *   Nmax     row pitch of AE_out in complex elements (>= every row's N)
 *   AE_out   [B][2][Nmax] complex128: element (b, ch, j) is the waveform at global bin kmin[b] + j, j < N_b;
 *            elements j >= N_b are left untouched
 *   kmin_out [B] int64, may be NULL
 */
int gb_waveform(gb_ctx *ctx, const double *params, int64_t B, int N, const int32_t *n_bins,
                int Nmax, double *AE_out, int64_t *kmin_out, void *stream);

/*
 * gb_delta_loglike -- delta lnL of B proposals (Eq. 4, Eq. 5).
 *   params_new   [B][8]; ADD: the proposed source; SWAP: the new source; REMOVE: ignored (may be NULL)
 *   params_old   [B][8]; REMOVE / SWAP: the source currently in the model; ADD: ignored (may be NULL)
 *   walker_index [B] int32 in [0, n_walkers)
 *   move         [B] int8 GB_ADD / GB_REMOVE / GB_SWAP, or NULL to use move_all for every row
 *   N, n_bins    as in gb_waveform (a SWAP row uses the same N for both sources)
 *   dlnL_out     [B] f64:  ADD <r|a> - <a|a>/2;  REMOVE -<r|h> - <h|h>/2;
 *                SWAP -( <a|a> + <o|o> - 2<a|o> - 2<r|a> + 2<r|o> ) / 2, <a|o> over the bins common to both windows
 *   aux_out      optional [B][2] f64: (<h|h>, <r|h>) of the new source (ADD, SWAP) or of the removed one
 */
int gb_delta_loglike(gb_ctx *ctx, const gb_data *data, const double *params_new, const double *params_old,
                     const int32_t *walker_index, const int8_t *move, int move_all, int N,
                     const int32_t *n_bins, int64_t B, double *dlnL_out, double *aux_out, void *stream);

/*
 * gb_residual_update -- scatter accepted moves into data->resid in place (Alg. 1) with
 * fp64 atomic adds: ADD r -= a; REMOVE r += h; SWAP r += o, r -= a.  accepted: [B] uint8 0/1, or NULL = all.
 * Rows that overlap in frequency within one walker are summed in an unspecified order (results differ from
 * a sequential sum by rounding only).
 */
int gb_residual_update(gb_ctx *ctx, const gb_data *data, const double *params_new, const double *params_old,
                       const int32_t *walker_index, const int8_t *move, int move_all, const uint8_t *accepted,
                       int N, const int32_t *n_bins, int64_t B, void *stream);

/*
 * Host-buffer forms (the end-to-end path): proposal arrays and outputs are HOST pointers (pinned memory
 * gives the best copy rate); `data` still describes DEVICE-resident residuals and PSDs, which are the state
 * that lives on the GPU across MCMC steps.  Each call copies its inputs to the device,
 * runs the device form on `stream`, copies the result back and synchronises `stream`.
 */
int gb_waveform_host(gb_ctx *ctx, const double *params /*HOST*/, int64_t B, int N, const int32_t *n_bins /*HOST*/,
                     int Nmax, double *AE_out /*HOST*/, int64_t *kmin_out /*HOST*/, void *stream);

int gb_delta_loglike_host(gb_ctx *ctx, const gb_data *data, const double *params_new /*HOST*/,
                          const double *params_old /*HOST*/, const int32_t *walker_index /*HOST*/,
                          const int8_t *move /*HOST*/, int move_all, int N, const int32_t *n_bins /*HOST*/,
                          int64_t B, double *dlnL_out /*HOST*/, double *aux_out /*HOST*/, void *stream);

/* gb_delta_loglike_accept (below) with HOST proposal arrays and HOST outputs; batches of >= 2^18 rows flow through in
 * 4 chunks, rows [B a_c / 24, B a_(c+1) / 24) with a = 0, 2, 9, 16, 24 (GB_HOST_ACCEPT_CUTS; the first chunk is the small one
 * because its copy is the only one no kernel hides).  Each chunk is one gb_delta_loglike_accept call: the snapshot
 * semantics hold per chunk, and a walker's rows should not straddle chunks if its accepted rows overlap.  apply = 0 runs
 * as a single chunk. */
#define GB_HOST_ACCEPT_CUTS {0, 2, 9, 16, 24}
int gb_delta_loglike_accept_host(gb_ctx *ctx, const gb_data *data, const double *params_new /*HOST*/,
                                 const double *params_old /*HOST*/, const int32_t *walker_index /*HOST*/,
                                 const int8_t *move /*HOST*/, int move_all, int N, const int32_t *n_bins /*HOST*/, int64_t B,
                                 const double *logq /*HOST*/, const double *logu /*HOST*/, const double *beta /*HOST*/,
                                 int64_t store_bins, int apply, double *dlnL_out /*HOST*/, double *aux_out /*HOST*/,
                                 uint8_t *accepted_out /*HOST*/, void *stream);

int gb_residual_update_host(gb_ctx *ctx, const gb_data *data, const double *params_new /*HOST*/,
                            const double *params_old /*HOST*/, const int32_t *walker_index /*HOST*/,
                            const int8_t *move /*HOST*/, int move_all, const uint8_t *accepted /*HOST*/,
                            int N, const int32_t *n_bins /*HOST*/, int64_t B, void *stream);

/*
 * gb_delta_loglike_keep / gb_residual_update_kept -- the sweep pair "delta lnL of every source, then scatter of the accepted
 * ones" (BASELINE config 5; Alg. 1 PAPER.md:599-613 in batched form) without generating the accepted waveforms twice.
 * gb_delta_loglike_keep is gb_delta_loglike for ADD / REMOVE rows (a SWAP row is a row error) that also writes every row's
 * window into context-owned scratch (2 x 16 bytes x sum_n_bins; DRAM is nearly idle under the compute-bound delta-lnL
 * kernels, so the stores are almost free on a B200).  sum_n_bins = sum of the rows' window lengths when n_bins is given
 * (ignored otherwise); too small a value sets row-error flag 4.
 * gb_residual_update_kept must be the next call on the context after gb_delta_loglike_keep (any other gb_* call except
 * gb_check / gb_band_sweep / gb_temper_sweep invalidates the kept state -> GB_ERR_INVALID).  It applies the moves of the
 * rows with accepted[b] != 0 (NULL: all rows) from the kept windows: ADD r -= a, REMOVE r += h; negate != 0 applies the
 * opposite signs (undo).  It may be called more than once.  Same result as gb_residual_update to the rounding order of
 * the atomics.  Both asynchronous on `stream`.
 */
int gb_delta_loglike_keep(gb_ctx *ctx, const gb_data *data, const double *params_new, const double *params_old,
                          const int32_t *walker_index, const int8_t *move, int move_all, int N, const int32_t *n_bins,
                          int64_t B, int64_t sum_n_bins, double *dlnL_out, double *aux_out, void *stream);
int gb_residual_update_kept(gb_ctx *ctx, const gb_data *data, const uint8_t *accepted, int negate, void *stream);

/*
 * gb_delta_loglike_accept -- the batched sweep step with its accept / reject decision (BASELINE config 5; acceptance of
 * Algorithm 1, with Eq. 13, in log form and the tempered likelihood of PAPER.md:674):
 *   1. delta lnL of every ADD / REMOVE row against the same residual snapshot, exactly as gb_delta_loglike
 *      (a SWAP row is a row error);
 *   2. row b is accepted iff  beta[b] * dlnL[b] + logq[b] >= logu[b]  (each operation rounded on its own; logq NULL: 0,
 *      beta NULL: 1; a NaN dlnL is rejected), written to accepted_out[b];
 *   3. apply != 0: the accepted rows update data->resid (ADD r -= a, REMOVE r += h) -- same result as
 *      gb_residual_update(accepted_out) after the call, to the rounding order of the atomics.
 * Only the ACCEPTED windows are kept (context-owned scratch of 32 bytes x store_bins, plus a few per cent of reservation
 * slack for batches of >= 2^18 rows; store_bins >= the sum of the accepted rows' window lengths, e.g. 0.3 x sum of n_bins
 * for a 25 % acceptance rate; a row that no longer fits is reported rejected and sets row-error flag 4), so no waveform is
 * generated twice and the scratch is a quarter of gb_delta_loglike_keep's.
 *   apply = 0   decide and keep; gb_residual_update_kept(ctx, data, NULL, negate, stream) applies (or undoes) the
 *               decisions later, any number of times, until the next gb_* call other than gb_check
 *   apply = 1   fused: batches of >= 2^19 rows are worked through in up to 8 chunks of WALKERS (geometrically shrinking);
 *               while chunk c + 1 is evaluated, the CTAs of the delta-lnL kernels move the accepted windows of chunks <= c
 *               -- complete, and read by no row any more, because rows of other walkers never read that residual -- from
 *               the store into the residual with bulk asynchronous copies and bulk add.f64 reductions (no thread waits
 *               for them), so the memory-bound update runs underneath the compute-bound evaluation and the snapshot
 *               semantics of step 1 hold exactly; a closing launch scatters what the last chunk accepted.  Smaller
 *               batches: as apply = 2
 *   apply = 2   the same decisions, the update as a separate launch after all evaluations
 *               (after apply = 1 or 2 the accepted windows stay in the context like after apply = 0:
 *               gb_residual_update_kept(ctx, data, NULL, 1, stream) undoes the call's update, e.g. for a step that the
 *               caller rejects as a whole; with negate = 0 it would apply the rows a second time)
 *   logq, logu, beta   [B] DEVICE f64 (logq, beta may be NULL);  accepted_out [B] DEVICE uint8;  dlnL_out, aux_out as
 *               gb_delta_loglike.  Asynchronous on `stream`.
 */
int gb_delta_loglike_accept(gb_ctx *ctx, const gb_data *data, const double *params_new, const double *params_old,
                            const int32_t *walker_index, const int8_t *move, int move_all, int N, const int32_t *n_bins,
                            int64_t B, const double *logq, const double *logu, const double *beta, int64_t store_bins,
                            int apply, double *dlnL_out, double *aux_out, uint8_t *accepted_out, void *stream);

/*
 * gb_overlap -- normalised overlap of B source pairs (cataloging; the search / catalog workloads
 * of PAPER.md:710-718 use the same kernels with this batch shape):
 *     O_b = <a_b|c_b> / sqrt(<a_b|a_b> <c_b|c_b>),   Eq. 2 against PSD row psd_row[b],
 * <a|c> over the bins common to the two windows, every term over the stored band only; O_b = 0 if a norm vanishes.
 *   data        only psd, psd_is_inverse, n_psd, k_lo, n_f are used (resid may be NULL)
 *   params_a, params_c  [B][8] DEVICE;  psd_row [B] DEVICE int32 or NULL (row 0)
 *   overlap_out [B] DEVICE f64;  aux_out optional [B][2] DEVICE: <a|a>, <c|c> (the optimal SNR^2 of each source)
 * N / n_bins as for gb_waveform.  Asynchronous on `stream`; a bad row sets the sticky flag and gives NaN.
 */
int gb_overlap(gb_ctx *ctx, const gb_data *data, const double *params_a, const double *params_c, const int32_t *psd_row,
               int N, const int32_t *n_bins, int64_t B, double *overlap_out, double *aux_out, void *stream);

/*
 * gb_band_sweep -- Algorithm 1 of the paper ("Galaxy sampling algorithm"): for each band task the
 * walker's residual on the staged bins is held on chip and the task's proposals are applied IN ORDER, each one a swap
 * theta_k -> theta'_k evaluated by Eq. 5 against the staged residual r', accepted iff
 *     beta * dlnL + logq >= logu          (Eq. 13, in log form; tempering PAPER.md:674)
 * and, when accepted, r' <- r' + h(theta_k) - h(theta'_k), theta_j[k] <- theta'_k.  The random
 * numbers of the method are inputs: logu = log of the uniform draw, logq = log prior / proposal-density ratio of the
 * proposal (0 for a symmetric in-model move); proposal generation (stretch / group / RJ) is
 * the caller's.  An RJ add or remove is the paper's amplitude switch: amp = 0 on one side.
 *
 *   tasks        [n_tasks] DEVICE array of gb_band_task
 *   N            window length of every source in this call (128, 256, 512, 1024); group bands by N
 *   max_stage    >= every task's n_stage, <= GB_BAND_MAX_STAGE; sizes the on-chip staging area
 *   params       [sum n_src][8] DEVICE, in/out: the current sources of every band (task i owns rows
 *                src_begin .. src_begin + n_src)
 *   prop_k       [sum n_prop] DEVICE int32: which source of its band proposal p replaces (0 .. n_src-1)
 *   prop_params  [sum n_prop][8], prop_logq [sum n_prop], prop_logu [sum n_prop]   DEVICE f64
 *   accepted_out [sum n_prop] DEVICE uint8, dlnL_out [sum n_prop] DEVICE f64 (the T = 1 delta lnL of every proposal)
 * Inner products use only the staged bins that lie in the stored band.  With GB_BAND_WRITE_BACK every accepted change
 * is also added to data->resid with FP64 atomics, so concurrent tasks of one walker must not propose into the same
 * bins: the paper's odd/even sub-band schedule -- one call per parity -- guarantees it.  Tasks are
 * independent and run concurrently; the proposals of one task run sequentially.
 * The library keeps the windows of each running task's current sources in context-owned scratch (about 150 MB, allocated at
 * the first call and kept), so that a proposal generates only the proposed waveform.
 * Errors: GB_ERR_INVALID for bad arguments; a task with a bad walker / n_stage or a proposal with a bad prop_k sets
 * the sticky row flag (gb_check) and gives NaN.  Asynchronous on `stream`.
 */
#define GB_BAND_MAX_STAGE 3072
/* task flags.  The last two implement the paper's odd/even cold-chain buffers (Fig. 4): per walker
 * only two residual rows are stored -- the data minus the cold-chain sources of the even sub-bands, and of the odd ones --
 * instead of one row per (temperature, walker).  A task of an odd sub-band stages from the EVEN row, which holds none of
 * the band's own sources, subtracts the band's current sources while staging (GB_BAND_SUBTRACT_CURRENT),
 * and, for the cold chain only, writes its accepted changes into the ODD row (GB_BAND_WRITE_OTHER); even
 * sub-bands the other way round.  Hotter chains stage from the same cold-chain row and write nothing. */
#define GB_BAND_WRITE_BACK 1        /* accepted changes are added to a stored residual row                      */
#define GB_BAND_SUBTRACT_CURRENT 2  /* r' = staged row - sum of the band's current sources (formed on chip)      */
#define GB_BAND_WRITE_OTHER 4       /* the write-back row is write_walker instead of walker                      */
typedef struct {
    int32_t walker;      /* residual row                                                        */
    int32_t n_src;       /* g_j: sources of the band                                            */
    int32_t src_begin;   /* first row of the band in params                                     */
    int32_t n_prop;      /* proposals of the band                                               */
    int32_t prop_begin;  /* first row of the band in prop_*                                     */
    int32_t n_stage;     /* staged bins                                                         */
    int64_t k_first;     /* global bin of staged bin 0                                          */
    int32_t flags;       /* GB_BAND_WRITE_BACK | GB_BAND_SUBTRACT_CURRENT | GB_BAND_WRITE_OTHER   */
    int32_t write_walker;/* residual row that receives accepted changes when GB_BAND_WRITE_OTHER */
    double beta;         /* inverse temperature of the band's chain                             */
} gb_band_task;
int gb_band_sweep(gb_ctx *ctx, const gb_data *data, const gb_band_task *tasks, int64_t n_tasks, int N, int max_stage,
                  double *params, const int32_t *prop_k, const double *prop_params, const double *prop_logq,
                  const double *prop_logu, uint8_t *accepted_out, double *dlnL_out, void *stream);

/*
 * gb_band_sweep_static -- gb_band_sweep (Algorithm 1) for callers that cannot allocate device memory
 * around the call: code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.  Same arguments,
 * same kernel, same results as gb_band_sweep; the only scratch of that kernel, the per-CTA cache of the current sources'
 * windows, lives in a file-scope device array of GB_STATIC_SCRATCH_BYTES (32 MiB) that every GPU which loads the library
 * holds until exit, and the call performs no cudaMalloc, no cudaFree and no allocating library call (gb_create, the
 * set-up, resolves the array's device address once per device).
 *   limit     n_tasks * N <= GB_STATIC_MAX_TASK_BINS (256 tasks of N = 128 ... 32 of N = 1024: one resident CTA and one
 *             32-window cache per task); a larger call returns GB_ERR_INVALID with the limit in gb_last_error and does
 *             nothing -- use gb_band_sweep
 *   sharing   every call on a device -- of every context -- uses the same array.  Nothing in it has to start at zero (a
 *             CTA writes a cache slot before it reads it, so the contents an earlier call left are never read) and
 *             nothing is cleared.  Calls that may OVERLAP on the GPU (different streams, or different contexts on one
 *             device) race on it: issue them on one stream or order them with events.
 * Asynchronous on `stream`; errors, flags and outputs as gb_band_sweep.
 */
#define GB_STATIC_SCRATCH_BYTES (32 * 1024 * 1024)
#define GB_STATIC_MAX_TASK_BINS 32768
int gb_band_sweep_static(gb_ctx *ctx, const gb_data *data, const gb_band_task *tasks, int64_t n_tasks, int N,
                         int max_stage, double *params, const int32_t *prop_k, const double *prop_params,
                         const double *prop_logq, const double *prop_logu, uint8_t *accepted_out, double *dlnL_out,
                         void *stream);

/*
 * gb_band_sweep_generate -- Algorithm 1 exactly as printed: the proposal step runs INSIDE the sequential
 * loop of each band, "k <- randint(0, g_j)", "theta'_k <- Make Proposal on theta", from the CURRENT
 * theta_k -- a stretch proposal built by the caller beforehand would use a stale theta_k as soon as an earlier proposal of
 * the same source was accepted.  The proposal is the group stretch of App. B with the stretch move of
 * Eq. 14:
 *   random numbers   Philox4x32-10, key = seed, counter = (proposal row, 0, block, sweep); block 0 -> k, friend, z;
 *                    block 1 -> the uniform of the accept step.  Results do not depend on how tasks are scheduled.
 *   k                floor(w0 g_j / 2^32);  uniforms u = (a + 1/2) 2^-52 from the top 26 bits of two words
 *   friends          `group` is the stationary group sorted by f0 ascending; the n_friends rows closest in
 *                    f0 to the current theta_k are a run of consecutive rows (ties: the lower rows); the auxiliary point is
 *                    row floor(w1 n_friends / 2^32) of that run
 *   z                g(z) ~ 1/sqrt(z) on [1/a, a]:  z = ((a - 1) u + 1)^2 / a
 *   theta'           theta_aux + z (theta_k - theta_aux) on all 8 coordinates; logq = 7 ln z (the z^(D-1) factor)
 *   periodic / prior coordinates flagged periodic are wrapped into [lo, hi); a proposal outside the box [lo, hi], or one
 *                    whose window [kmin', kmin' + N) leaves the task's staged bins ("we allow samples to go halfway into
 *                    neighboring bands"), has zero prior: rejected without a likelihood evaluation, dlnL = NaN
 *   accept           beta * dlnL + logq >= logu with logu = ln(uniform of block 1), as gb_band_sweep
 * Everything else (staging, Eq. 5, updates, write-back, task flags, errors) is gb_band_sweep.  A task needs n_src >= 1
 * and n_stage >= 1.  Outputs per proposal row, all DEVICE: k_out int32, params_out [.][8], logq_out, logu_out (what was
 * generated), accepted_out, dlnL_out.  k and theta' are reproducible bit for bit from the definition above.
 */
typedef struct {             /* HOST POD */
    uint64_t seed;           /* Philox key                                                         */
    uint32_t sweep;          /* counter word 3: a new value for every call of a run                 */
    int32_t n_friends;       /* size of the friends run (clamped to n_group)                        */
    const double *group;     /* DEVICE [n_group][8] parameter rows sorted by f0 (column 1) ascending */
    int64_t n_group;
    double stretch_a;        /* a > 1 (2 in ref. [59] of the paper)                                 */
    double lo[8], hi[8];     /* prior box per coordinate                                            */
    int32_t periodic[8];     /* != 0: coordinate wrapped into [lo, hi)                              */
} gb_stretch;
int gb_band_sweep_generate(gb_ctx *ctx, const gb_data *data, const gb_band_task *tasks, int64_t n_tasks, int N,
                           int max_stage, double *params, const gb_stretch *gen, int32_t *k_out, double *params_out,
                           double *logq_out, double *logu_out, uint8_t *accepted_out, double *dlnL_out, void *stream);

/*
 * gb_temper_sweep -- Algorithm 2 of the paper ("Galaxy Tempering algorithm") with the swap acceptance
 * of Eq. D2 for walkers that carry different residuals / PSDs.  One task = one sub-band with a ladder of
 * n_t chains (n_t <= GB_TEMPER_MAX_LADDER); chain entry c = chain_begin + t has
 *   chain_walker[c]     residual row of chain t (the paper's permuted walker p[t]; r = d - H of that chain)
 *   chain_beta[c]       inverse temperature
 *   chain_set_begin[c], chain_set_n[c]   the band's sources the chain holds at entry: rows of params (read-only)
 *   chain_logu[c]       log of the uniform draw of the pair (t, t-1); entry t = 0 unused
 * From t = n_t - 1 down to 1 chains i = t and j = t - 1 propose to exchange the sets S_i, S_j they currently hold.  With
 * delta = sum_{S_i} h - sum_{S_j} h on the staged bins,  D_i = lnL_i(S_j) - lnL_i(S_i) = -1/2 <delta|delta>_i - <r_i|delta>_i,
 * D_j = lnL_j(S_i) - lnL_j(S_j) = -1/2 <delta|delta>_j + <r_j|delta>_j  (each chain's own PSD row), accepted iff
 * beta_i D_i + beta_j D_j >= logu.  Accepted: the holders are exchanged and, if write_back, r_i += delta, r_j -= delta in
 * data->resid (FP64 atomics; the paper keeps only the cold chain's residual, here every chain owns one).
 * Ladders of up to 32 chains sum each chain's set once into context-owned scratch (allocated at the first call, <= 700 MB).
 * Outputs [n_chain]: perm_out[c] = ladder position whose INITIAL set ends in chain t; accepted_out[c]; dlnl_out[c][2] =
 * (D_i, D_j) of pair (t, t-1).  All arrays DEVICE.  N, max_stage, odd/even rule, errors and asynchrony as gb_band_sweep.
 *
 * Odd/even cold-chain buffers (Algorithm 2 as printed): with GB_TEMPER_ODD_EVEN the
 * row of a chain's walker is the opposite-parity cold-chain buffer, which holds none of the band's own sources, so the
 * kernel forms each chain's residual on chip, r_t = row(chain_walker[t]) - sum_{S_t} h over the set the chain holds
 * (PAPER.md:626-631), and only an exchange with the cold chain (pair (1, 0)) is written: -delta into
 * row write_walker, the cold chain's buffer of the band's own parity.  Ladders of up to GB_TEMPER_MAX_LADDER_ODD_EVEN
 * chains (a longer one is a row error).  This is the mode that composes with gb_band_sweep's GB_BAND_SUBTRACT_CURRENT /
 * GB_BAND_WRITE_OTHER: both then work on the 2 x n_walkers rows of the odd/even layout.
 */
#define GB_TEMPER_MAX_LADDER 64
#define GB_TEMPER_MAX_LADDER_ODD_EVEN 32
#define GB_TEMPER_WRITE_BACK 1   /* accepted exchanges update data->resid                                           */
#define GB_TEMPER_ODD_EVEN 2     /* rows hold none of the band's sources; write only the cold chain, to write_walker */
typedef struct {
    int32_t n_t;          /* chains of the ladder                    */
    int32_t chain_begin;  /* first chain entry of the task           */
    int32_t n_stage;      /* staged bins                             */
    int32_t write_back;   /* GB_TEMPER_WRITE_BACK | GB_TEMPER_ODD_EVEN */
    int64_t k_first;      /* global bin of staged bin 0              */
    int32_t write_walker; /* GB_TEMPER_ODD_EVEN: row that receives exchanges with the cold chain */
    int32_t reserved;     /* set to 0                                */
} gb_temper_task;
int gb_temper_sweep(gb_ctx *ctx, const gb_data *data, const gb_temper_task *tasks, int64_t n_tasks, int N, int max_stage,
                    const double *params, const int32_t *chain_walker, const double *chain_beta,
                    const int32_t *chain_set_begin, const int32_t *chain_set_n, const double *chain_logu,
                    int32_t *perm_out, uint8_t *accepted_out, double *dlnl_out, void *stream);

#ifdef __cplusplus
}
#endif
#endif /* GBFIT_H */
