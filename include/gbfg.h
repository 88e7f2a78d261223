/* gbfg.h — C ABI of libgbfg, the B200 (sm_100a) galactic-binary foreground simulator.
 *
 * What the library computes: catalog of galactic binaries (A, f, fdot per source) ->
 * confusion-noise power spectral density S_n(f) by the iterative subtraction algorithm of
 * arxiv 2602.18560, Appendix D (steps 1-10 at :521-530), in the power-domain
 * form of BASELINE.json:configs[0].  DESIGN.md §3 (R0-R6) states every reading of the paper that
 * the arithmetic below follows; DESIGN.md §4 specifies the elementary functions of stage (i).
 *
 * Conventions
 *  - "dev" pointers are DEVICE pointers owned by the caller (e.g. torch tensors); "host" pointers
 *    are ordinary host memory.  The library never frees or retains a caller pointer past the
 *    call, except that asynchronous calls use them until the work queued on `stream` has run.
 *  - `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).
 *  - Catalogs are structure-of-arrays binary64: A[N], f[N], fdot[N].  A batch of n_cat catalogs is
 *    the concatenation of its catalogs; `offsets` (HOST, n_cat+1 entries, offsets[0] = 0) gives the
 *    first source of each.  Per-bin arrays of a batch are [n_cat][n_bins], row-major.
 *  - The spectrum is int64 fixed point: one unit = 2^scale_log2 strain^2 (configs: -140).
 *  - A `workspace` is DEVICE memory, 32-byte aligned (cudaMalloc gives 256), of at least gbfg_workspace_bytes();
 *    GBFG_ERR_WORKSPACE otherwise.
 *  - Every function returns GBFG_OK (0) or a negative gbfg_status.  Nothing throws, aborts or
 *    prints.  The four stage calls and the helpers are asynchronous on `stream`;
 *    gbfg_subtract_until_converged and gbfg_simulate* wait, once per iteration, for that iteration's block of
 *    counters (selected and near-threshold sources per catalog, flags: a few dozen int64 the device stores into
 *    mapped pinned host memory, R9), synchronise `stream` before they return and fill HOST results.
 *  - What the library keeps between calls is per host thread and belongs to the device that was current when it
 *    was made (a side stream, a few events, gbfg_simulate_host's device arena); a thread that calls again with
 *    another current device gets fresh ones.  An error return leaves no work of the call in flight.
 *  - The library runs on compute capability 10.x devices only (GBFG_ERR_ARCH otherwise).  There is
 *    no CPU fallback and no other backend.
 */
#ifndef GBFG_H
#define GBFG_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum gbfg_status {
    GBFG_OK = 0,
    GBFG_ERR_INVALID_ARG = -1, /* null pointer, even / non-positive window, n_bins < h+1, f_min >= f_max, bad struct_size, n_cat out of range */
    GBFG_ERR_WORKSPACE = -2,   /* workspace NULL, not aligned or smaller than gbfg_workspace_bytes() */
    GBFG_ERR_CUDA = -3,        /* a CUDA runtime call failed: see gbfg_last_cuda_error() */
    GBFG_ERR_ARCH = -4,        /* current device is not compute capability 10.x */
    GBFG_ERR_UNSUPPORTED = -5, /* window wider than GBFG_MAX_WINDOW, n_cat > GBFG_MAX_CAT, alpha_gamma outside its stated range */
    GBFG_ERR_STATIC_LIMIT = -6 /* gbfg_running_median_static: the call needs more scratch than GBFG_STATIC_SCRATCH_BYTES */
} gbfg_status;

#define GBFG_MAX_CAT 256        /* catalogs per batched call */
#define GBFG_MAX_WINDOW 4097    /* widest running-median window of this build (odd) */
#define GBFG_MAX_ITER_TRACE 64  /* per-iteration counts kept in gbfg_iter_result */
#define GBFG_PAPER_ALPHA_MIN 0.25   /* range of gbfg_pop_paper.alpha_gamma the special functions of DESIGN.md R12 are */
#define GBFG_PAPER_ALPHA_MAX 16.0   /* stated and pinned for (Table I, draws it from [1, 3]) */

/* Frequency grid: bins of width 1/t_obs covering [f_min, f_max); bin k = [f_min + k/T, f_min + (k+1)/T).
 * n_bins = ceil((f_max - f_min) * t_obs)  (R2).  Fill with gbfg_grid_init. */
typedef struct gbfg_grid {
    uint32_t struct_size;   /* = sizeof(gbfg_grid) */
    int32_t scale_log2;     /* spectrum unit = 2^scale_log2 */
    double f_min, f_max;    /* Hz */
    double t_obs;           /* s */
    int64_t n_bins;
} gbfg_grid;

/* Population parameters Lambda of BASELINE.json's generator (configs[0], configs[4]):
 *   p(f) ∝ f^-slope on [f_min, f_max);  log10 A ~ N(logA_offset + (2/3) log10(f / 1 mHz), logA_sigma);
 *   fdot = (96/5) pi^(8/3) (G Mc / c^3)^(5/3) f^(11/3)  (eq. 4),
 *   log10(Mc / Msun) ~ N(logMc_mean, logMc_sigma). */
typedef struct gbfg_pop {
    uint32_t struct_size;   /* = sizeof(gbfg_pop) */
    uint32_t reserved;
    double slope, logA_offset, logA_sigma, logMc_mean, logMc_sigma;
    int64_t n_src;
} gbfg_pop;

/* Population parameters Lambda of the paper's own model, eq. (9) PAPER.md:126 (Table I; R12):
 *   p(f) ∝ f^alpha_pl on the grid's band;  log10(fdot / Hz s^-1) - mu_gamma ~ Gamma(alpha_gamma, rate beta_gamma) (eq. 7);
 *   log10[(f/Hz)^(-2/3) A] - mu ~ LogNormal(0, sigma) (eq. 8);  (f, fdot) tied by a Gaussian copula of correlation rho. */
typedef struct gbfg_pop_paper {
    uint32_t struct_size;   /* = sizeof(gbfg_pop_paper) */
    uint32_t reserved;
    double alpha_pl, alpha_gamma, beta_gamma, mu_gamma, mu, sigma, rho;
    int64_t n_src;
} gbfg_pop_paper;

/* Parameters of the subtraction loop (R3, R4, R6). */
typedef struct gbfg_iter_params {
    uint32_t struct_size;   /* = sizeof(gbfg_iter_params) */
    int32_t window;         /* odd running-median window W = 2h+1 (paper: ~2000) */
    double median_norm;     /* C of eq. (D3); paper value exactly 729/512 */
    double rho_th;          /* SNR threshold, 7 in the paper */
    int32_t max_iter;       /* iteration cap (BASELINE: 30) */
    uint32_t flags;         /* GBFG_FLAG_* */
    double psd_rtol;        /* > 0: also stop when the PSD has converged (R13): from the second
                               iteration on, max_k |S_n^(i)[k] - S_n^(i-1)[k]| / S_n^(i-1)[k] <= psd_rtol ends a catalog's
                               loop before that iteration's SNR test.  <= 0: off (the paper gives no tolerance) */
} gbfg_iter_params;

#define GBFG_FLAG_NO_PRESELECT 1u   /* test every unresolved source every iteration (no R5 candidate cut) */
#define GBFG_FLAG_NO_INCREMENTAL 2u /* recompute every median tile every iteration (no dirty-tile skipping) */
#define GBFG_FLAG_ESTIMATOR_MEAN 4u /* running mean, eq. (D1), instead of the running median (R8):
                                       dev_median receives the window sums, median_norm is not used */

/* Per-catalog outcome of the loop (HOST). */
typedef struct gbfg_iter_result {
    int32_t n_iter;             /* iterations run; = max_iter when the cap was hit */
    int32_t converged;          /* 1: an iteration resolved no new source; 2: the PSD converged (psd_rtol); 0: cap hit */
    int64_t n_resolved;         /* sources resolved by this call */
    int64_t n_near_threshold;   /* tests with |rho^2 / rho_th^2 - 1| <= 2e-9, summed over iterations */
    int64_t n_candidates;       /* sources that passed the pre-selection (= tested sources if disabled) */
    int64_t n_median_outputs;   /* running-median outputs computed, summed over iterations (n_bins per full pass) */
    int64_t n_snr_tests;        /* SNR tests evaluated, summed over iterations */
    int64_t n_new_per_iter[GBFG_MAX_ITER_TRACE];
} gbfg_iter_result;

int gbfg_version(void);                    /* 10000*major + 100*minor + patch */
const char *gbfg_strerror(int status);     /* static string */
const char *gbfg_last_cuda_error(void);    /* thread-local; text of the CUDA error behind the last GBFG_ERR_CUDA */

/* Fills *out, computing n_bins = ceil((f_max - f_min) * t_obs).  INVALID_ARG unless
 * 0 < f_min < f_max, t_obs > 0 and 1 <= n_bins < 2^31. */
int gbfg_grid_init(double f_min, double f_max, double t_obs, int32_t scale_log2, gbfg_grid *out);

/* Helper: Robson, Cornish & Liu 2019 sky-averaged LISA noise (paper ref [70]) with
 * BASELINE.json:configs[0]'s constants, evaluated at bin centres f_min + (k + 1/2)/T (R3).
 * dev_s_instr: [n_bins] binary64, written. */
int gbfg_instrument_noise(const gbfg_grid *grid, double *dev_s_instr, void *stream);

/* Helper: SciRDv1 noise of the TDI channels, eqs. (C1)-(C5), and its rescaling by the TDI
 * response, eqs. (B2)-(B5), at the bin centres (R11).  P_pm, A_fm: the OMS and
 * test-mass amplitudes in pm and fm s^-2 (SciRDv1: 15 and 3); L_m: arm length in metres; tdi2 != 0: TDI 2.0,
 * eq. (C5).  Written (each [n_bins] binary64, any may be NULL but not all): dev_S_AA = S^AA = S^EE (C3),
 * dev_S_TT (C4), dev_Sh_AA = S^AA / R_AA, dev_Sh_TT = S^TT / R_TT (B2: strain-equivalent noise, usable as the
 * s_instr of the stage calls). */
int gbfg_instrument_noise_aet(const gbfg_grid *grid, double P_pm, double A_fm, double L_m, int32_t tdi2,
                              double *dev_S_AA, double *dev_S_TT, double *dev_Sh_AA, double *dev_Sh_TT, void *stream);

/* Helper: the noise curve of the SNR summed over the TDI channels A, E, T, eq. (11), in the power domain
 * (R14): a source's strain power p enters channel X with the sky-averaged response R_XX, so the channel's term of
 * eq. (11) is 4 p / S_h^XX with S_h^XX = S^XX / R_XX (the dev_Sh_* outputs of gbfg_instrument_noise_aet); A and E are equal,
 * hence rho^2 = sum_bins 4 p / S_sum with  S_sum = 1 / ((2 / S_h^AA) + (1 / S_h^TT)).  Handing dev_Sh_sum to the stage calls as
 * their s_instr makes every SNR of the loop the channel-summed one.  All arrays [n_bins] binary64, DEVICE. */
int gbfg_channel_sum_noise(const double *dev_Sh_AA, const double *dev_Sh_TT, int64_t n_bins, double *dev_Sh_sum, void *stream);

/* Stage (i) — step 1 of the algorithm: draw every catalog of the batch from its
 * population with Philox4x32-10 (R1, §4).  pops: HOST [n_cat]; offsets: HOST [n_cat+1]
 * with offsets[c+1]-offsets[c] = pops[c].n_src.  Catalog c uses Philox counter word 3 =
 * first_cat_id + c, so a batch can be drawn in pieces.  dev_A / dev_f / dev_fdot: [offsets[n_cat]],
 * written (16-byte aligned). */
int gbfg_sample_catalog(const gbfg_grid *grid, const gbfg_pop *pops, const int64_t *offsets,
                        int32_t n_cat, uint32_t first_cat_id, uint64_t seed,
                        double *dev_A, double *dev_f, double *dev_fdot, void *stream);

/* Stage (i) with the paper's own population model (Table I, eqs. 7-9, Gaussian copula of Appendix A steps iii-iv,
 * PAPER.md:454-457; R12).  Same conventions as gbfg_sample_catalog (Philox counter blocks 2 and 3, so the two
 * samplers never share a random number); alpha_gamma, beta_gamma > 0, sigma >= 0, 0 <= rho < 1 (INVALID_ARG otherwise);
 * alpha_gamma outside [GBFG_PAPER_ALPHA_MIN, GBFG_PAPER_ALPHA_MAX]: GBFG_ERR_UNSUPPORTED. */
int gbfg_sample_catalog_paper(const gbfg_grid *grid, const gbfg_pop_paper *pops, const int64_t *offsets,
                              int32_t n_cat, uint32_t first_cat_id, uint64_t seed,
                              double *dev_A, double *dev_f, double *dev_fdot, void *stream);

/* Stage (ii)/(v) — deposit (sign = +1) or subtract (sign = -1) source power (R2;
 * subtraction is eq. (D4)): for every addressed source
 *     spectrum[c][k] += sign * q_i   for k in [k0_i, k0_i + w_eff_i).
 * dev_sel_idx == NULL: all sources.  Otherwise dev_sel_idx holds GLOBAL source indices and
 * dev_sel_count points to one int64 on the device = number of entries (read on the device).
 * dev_spectrum: [n_cat][n_bins] int64, accumulated into (zero it first for a fresh deposit).
 * dev_err_count: one int64, incremented by the number of rejected sources (NaN, A<0, fdot<0, f
 * outside the band: DOMAIN; width or quantised power beyond 2^62: RANGE); may be NULL.
 * workspace: >= gbfg_workspace_bytes(...); holds the difference array of the range-update form. */
int gbfg_deposit(const gbfg_grid *grid, const double *dev_A, const double *dev_f, const double *dev_fdot,
                 const int64_t *offsets, int32_t n_cat,
                 const int64_t *dev_sel_idx, const int64_t *dev_sel_count, int32_t sign,
                 int64_t *dev_spectrum, int64_t *dev_err_count,
                 void *workspace, size_t workspace_bytes, void *stream);

/* Stage (iii) — exact running median of eq. (D2), PAPER.md:542 (R3): for each row,
 * median_out[k] = the h-th smallest of x[k-h .. k+h], W = 2h+1 odd, ends reflected
 * (x[-j] = x[j-1], x[n-1+j] = x[n-j]).  Requires n_bins >= h+1 and W <= GBFG_MAX_WINDOW.
 * dev_spectrum, dev_median_out: [n_cat][n_bins] int64 (must not alias).
 * workspace: DEVICE, 16-byte aligned, >= gbfg_running_median_workspace_bytes(n_bins, n_cat, window) bytes (a workspace of
 * gbfg_workspace_bytes() for the same grid is large enough too); GBFG_ERR_WORKSPACE otherwise.  Nothing is allocated. */
int gbfg_running_median(const int64_t *dev_spectrum, int64_t n_bins, int32_t n_cat, int32_t window,
                        int64_t *dev_median_out, void *workspace, size_t workspace_bytes, void *stream);
size_t gbfg_running_median_workspace_bytes(int64_t n_bins, int32_t n_cat, int32_t window);   /* 0: invalid arguments */

/* gbfg_running_median for callers that must not allocate and have no workspace to hand in (CUDA graph capture, serving
 * loops, harnesses that forbid cudaMalloc): same operation, same arguments without the workspace, same results to the
 * bit.  The scratch the kernels need (the list of tiles the 32-bit-key kernel leaves to the 64-bit-key one: 256 bytes of
 * counters + 16 bytes per tile) lives in ONE array of GBFG_STATIC_SCRATCH_BYTES in the library's device image: every
 * device that loads the library holds it until the process exits.  A call that needs more (more than
 * GBFG_STATIC_MAX_TILES tiles over all rows; a tile is at most 8704 - (window - 1) outputs, so 4.3e8 outputs at
 * window 2001) returns GBFG_ERR_STATIC_LIMIT and launches nothing: use gbfg_running_median.  The call allocates nothing
 * (no cudaMalloc / cudaFree, no allocating library routine; the array's device address is looked up once per device).
 * The array is shared by every call and keeps the last call's contents; the counters are cleared on the stream at the
 * start of each call.  Calls that may OVERLAP on the GPU (two streams, two host threads, two captured graphs running
 * side by side) race on it: order them, or use gbfg_running_median with a workspace each. */
#define GBFG_STATIC_SCRATCH_BYTES (1 << 20)
#define GBFG_STATIC_MAX_TILES ((GBFG_STATIC_SCRATCH_BYTES - 256) / 16)
int gbfg_running_median_static(const int64_t *dev_spectrum, int64_t n_bins, int32_t n_cat, int32_t window,
                               int64_t *dev_median_out, void *stream);

/* Running-mean estimator of eq. (D1), PAPER.md:538 (the paper's production choice, :176, :552; R8):
 * sum_out[c][k] = sum of x[c][k-h .. k+h], W = 2h+1 odd, ends reflected as for the median (the exact
 * object is the int64 window sum; it must fit int64), and, when dev_psd != NULL,
 * psd[c][k] = s_instr[k] + (sum_out[c][k] * 2^scale_log2) / W   (eq. 10).  dev_s_instr and dev_psd are both
 * NULL or both given.  Same size limits as gbfg_running_median. */
int gbfg_running_mean(const int64_t *dev_spectrum, int64_t n_bins, int32_t n_cat, int32_t window,
                      int64_t *dev_sum_out, const double *dev_s_instr, int32_t scale_log2,
                      double *dev_psd, void *stream);

/* psd[c][k] = s_instr[k] + median_norm * (median[c][k] * 2^scale_log2): eqs. (10), (D2), (D3)
 * (PAPER.md:142-145, 542-549).  dev_s_instr: [n_bins], shared by the batch. */
int gbfg_psd(const int64_t *dev_median, const double *dev_s_instr, int64_t n_bins, int32_t n_cat,
             double median_norm, int32_t scale_log2, double *dev_psd, void *stream);

/* Coarse-graining of the PSD, eqs. (13)-(14), and the characteristic strain of eq. (B1)
 * (PAPER.md:465); R10.  dev_edges: DEVICE [n_coarse + 1] non-decreasing fine-bin indices; coarse bin k
 * holds the fine bins edges[k] <= i < edges[k+1] (clipped to [0, n_bins]), whose frequencies are the bin centres
 * f_min + (i + 1/2)/t_obs.  Written: dev_S [n_cat][n_coarse] = mean PSD of the bin (eq. 13), dev_f [n_coarse] =
 * mean frequency (eq. 14; may be NULL), dev_hc [n_cat][n_coarse] = sqrt(f S) (eq. B1; may be NULL).  An empty
 * coarse bin gives NaN.  The mean is within a few ulp of the exactly rounded one (compensated summation). */
int gbfg_coarse_grain(const double *dev_psd, int64_t n_bins, int32_t n_cat, const int64_t *dev_edges,
                      int32_t n_coarse, double f_min, double t_obs, double *dev_S, double *dev_f,
                      double *dev_hc, void *stream);

/* Stage (iv) — SNR of every unresolved source against the current PSD and selection
 * (eqs. 11-12; R4): rho2_i = sum_{k in bins(i)} 4 p_i / psd[c][k];
 * newly resolved iff rho2_i > rho_th^2 (strict).  For those, dev_resolved[i] is set to 1 and i is
 * appended to dev_sel_idx (set semantics: order unspecified).
 *  dev_resolved:  [N] uint8 in/out; sources with a non-zero flag are not tested.
 *  dev_rho2_out:  [N] or NULL; rho2 of every tested source (NaN for rejected sources); untested
 *                 entries are left untouched.
 *  dev_sel_idx:   [N] capacity, written.   dev_sel_count: [1 + n_cat] int64, written: total, then
 *                 the number selected in each catalog.
 *  dev_near_count: one int64 or NULL, incremented by the number of tests within 1e-9 (relative, in
 *                 rho) of the threshold. */
int gbfg_snr_select(const gbfg_grid *grid, const double *dev_A, const double *dev_f, const double *dev_fdot,
                    const int64_t *offsets, int32_t n_cat, const double *dev_psd, double rho_th,
                    uint8_t *dev_resolved, double *dev_rho2_out,
                    int64_t *dev_sel_idx, int64_t *dev_sel_count, int64_t *dev_near_count,
                    void *workspace, size_t workspace_bytes, void *stream);

/* Stage (v) — the loop, steps 4-10 (R6), device resident; the host reads one small
 * block of counters per iteration (see Conventions).  Catalogs of a batch iterate independently; a catalog
 * that resolved nothing is frozen.
 *  dev_spectrum: [n_cat][n_bins] in: total deposited spectrum, out: residual.
 *  dev_median, dev_psd: [n_cat][n_bins] out, always those of the returned residual.
 *  dev_resolved: [N] uint8 in/out (zero it for a fresh run).
 *  host_results: HOST [n_cat]. */
int gbfg_subtract_until_converged(const gbfg_grid *grid, const double *dev_A, const double *dev_f,
                                  const double *dev_fdot, const int64_t *offsets, int32_t n_cat,
                                  const double *dev_s_instr, const gbfg_iter_params *params,
                                  int64_t *dev_spectrum, int64_t *dev_median, double *dev_psd,
                                  uint8_t *dev_resolved, gbfg_iter_result *host_results,
                                  void *workspace, size_t workspace_bytes, void *stream);

/* The whole hot path on device buffers: sample (i) -> deposit (ii) -> loop (iii)-(v).
 * Outputs as above plus the catalog itself and the total spectrum (dev_total may be NULL).
 * dev_err_count: one int64 or NULL.
 * cat_ids: HOST [n_cat] or NULL.  Philox counter word 3 of catalog c (R1) is cat_ids[c], or c when NULL:
 * a rank that runs a share {c_0, c_1, ...} of a batch (any subset, any order) passes those ids and
 * gets, row by row, the bits the whole batch gives for those catalogs. */
int gbfg_simulate(const gbfg_grid *grid, const gbfg_pop *pops, const int64_t *offsets, int32_t n_cat,
                  uint64_t seed, const uint32_t *cat_ids, const double *dev_s_instr, const gbfg_iter_params *params,
                  double *dev_A, double *dev_f, double *dev_fdot,
                  int64_t *dev_total, int64_t *dev_spectrum, int64_t *dev_median, double *dev_psd,
                  uint8_t *dev_resolved, int64_t *dev_err_count, gbfg_iter_result *host_results,
                  void *workspace, size_t workspace_bytes, void *stream);

/* The path as the paper runs it (Fig. 3): the paper's own population model (gbfg_pop_paper, Table I)
 * -> catalog -> deposit -> loop -> optionally the coarse-grained S_n, mean frequencies and h_c of eqs. (13)-(14), (B1)
 * (dev_edges / n_coarse / dev_S_coarse / dev_f_coarse / dev_hc as for gbfg_coarse_grain; dev_edges = dev_S_coarse = NULL:
 * no epilogue).  The paper's production settings are params->flags = GBFG_FLAG_ESTIMATOR_MEAN (eq. D1) and a psd_rtol > 0
 * (PAPER.md:530, 552).  Everything else as gbfg_simulate. */
int gbfg_simulate_paper(const gbfg_grid *grid, const gbfg_pop_paper *pops, const int64_t *offsets, int32_t n_cat,
                        uint64_t seed, const uint32_t *cat_ids, const double *dev_s_instr, const gbfg_iter_params *params,
                        double *dev_A, double *dev_f, double *dev_fdot,
                        int64_t *dev_total, int64_t *dev_spectrum, int64_t *dev_median, double *dev_psd,
                        uint8_t *dev_resolved, int64_t *dev_err_count, gbfg_iter_result *host_results,
                        const int64_t *dev_edges, int32_t n_coarse, double *dev_S_coarse, double *dev_f_coarse, double *dev_hc,
                        void *workspace, size_t workspace_bytes, void *stream);

/* The same path with HOST buffers: the library allocates device memory, copies host_s_instr in,
 * runs gbfg_simulate on its own stream, and copies the PSD ([n_cat][n_bins] binary64) and the
 * resolved flags ([N] uint8, may be NULL) back.  host_s_instr == NULL: the curve of gbfg_instrument_noise
 * (a function of the grid alone) is made on the device instead of being uploaded.  Host pointers should be
 * pinned for full speed; with a pinned host_psd the PSD leaves for the host while the loop still runs (blocks
 * that change afterwards are stored again: every bin arrives with its final value).
 * Synchronous.  The device memory it allocates is cached per host thread (gbfg_release_cached). */
int gbfg_simulate_host(const gbfg_grid *grid, const gbfg_pop *pops, const int64_t *offsets, int32_t n_cat,
                       uint64_t seed, const uint32_t *cat_ids, const double *host_s_instr, const gbfg_iter_params *params,
                       double *host_psd, uint8_t *host_resolved, gbfg_iter_result *host_results);

/* gbfg_simulate_host keeps its device arena and stream between calls of the same host thread, so that
 * repeated calls do not pay cudaMalloc / cudaFree; this frees them (synchronises the stream first), together with
 * the side stream and events the loop keeps per host thread. */
int gbfg_release_cached(void);

/* Bytes of device workspace sufficient for any call above on this grid / batch. */
size_t gbfg_workspace_bytes(const gbfg_grid *grid, int64_t n_src_total, int32_t n_cat);

/* Number of kernels the calling thread's library calls have launched so far (for bench.py). */
int64_t gbfg_kernel_launch_count(void);

/* Measurement helper (bench.py's roofline leg).  While enabled for the calling
 * thread, every kernel the library launches is bracketed by a pair of CUDA events recorded on the
 * stream the kernel is launched on.  gbfg_profile_read waits for those events, fills
 * out[GBFG_K_*] (HOST, n_out >= GBFG_K_COUNT) with the number of timed launches of each kernel
 * class and their summed / largest device time in milliseconds, and clears the record.
 * Costs two event records per launch; off by default. */
enum {
    GBFG_K_SAMPLE = 0,      /* sample_kernel                      stage (i)   */
    GBFG_K_NOISE,           /* instrument_noise_kernel            helper      */
    GBFG_K_DEPOSIT,         /* deposit kernels                    stage (ii)/(v) */
    GBFG_K_SCAN,            /* difference-array scan kernels      stage (ii)/(v) */
    GBFG_K_MEDIAN,          /* running median (+ fused PSD)       stage (iii) */
    GBFG_K_PSD,             /* psd_kernel                         stage (iii) */
    GBFG_K_INV_BLOCKS,      /* block sums of 1/psd                stage (iv)  */
    GBFG_K_SNR,             /* SNR + select kernels               stage (iv)  */
    GBFG_K_AUX,             /* plan_kernel: dirty blocks -> median work list  */
    GBFG_K_COUNT
};
typedef struct gbfg_kernel_time {
    int64_t launches;
    double total_ms;
    double max_ms;
} gbfg_kernel_time;
int gbfg_profile_enable(int on);
int gbfg_profile_read(gbfg_kernel_time *out, int32_t n_out);
/* The same record launch by launch, in the order the launches were issued: kernel class, start and end of each timed
 * launch in milliseconds since the first one's start (launches on different streams overlap).  out: HOST, room for cap
 * entries; *n_written = the number filled (at most cap; *n_total = the number recorded).  Does not clear the record:
 * gbfg_profile_read or gbfg_profile_enable does. */
typedef struct gbfg_launch_time {
    int32_t kernel;         /* GBFG_K_* */
    float start_ms, end_ms;
} gbfg_launch_time;
int gbfg_profile_timeline(gbfg_launch_time *out, int32_t cap, int32_t *n_written, int32_t *n_total);

#ifdef __cplusplus
}
#endif
#endif /* GBFG_H */
