// gbfg_common.cuh — shared declarations of the CUDA side of libgbfg (sm_100a).
//
// Nothing in this directory is shared with oracle/: constants and algorithms are typed here
// independently from DESIGN.md §3-§4.  The translation units are compiled with -fmad=false so
// that every binary64 operation is singly rounded; fma() appears only where DESIGN.md §4 says so.
#pragma once

#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>

#include "../../include/gbfg.h"

namespace gbfg {

// ---------------------------------------------------------------------------------------------
// host-side plumbing
// ---------------------------------------------------------------------------------------------
int set_cuda_error(cudaError_t e, const char *where);   // records text, returns GBFG_ERR_CUDA
int check_device();                                     // GBFG_OK or GBFG_ERR_ARCH / GBFG_ERR_CUDA
void count_launch(int n = 1);
int sm_count();
// stage (i) with explicit catalog ids (sample.cu): cat_ids HOST [n_cat] or NULL (first_cat_id + c)
int sample_catalog_paper_ids(const gbfg_grid *grid, const gbfg_pop_paper *pops, const int64_t *offsets, int32_t n_cat,
                             uint32_t first_cat_id, const uint32_t *cat_ids, uint64_t seed,
                             double *dev_A, double *dev_f, double *dev_fdot, void *stream);
struct SampleDeposit;       // != NULL: every source is also deposited by the kernel that draws it (gbfg_simulate)
int sample_catalog_ids(const gbfg_grid *grid, const gbfg_pop *pops, const int64_t *offsets, int32_t n_cat,
                       uint32_t first_cat_id, const uint32_t *cat_ids, uint64_t seed,
                       double *dev_A, double *dev_f, double *dev_fdot, void *stream, const SampleDeposit *dep = nullptr);

// Kernel classes of the per-kernel timing helper (gbfg_profile_*; order = GBFG_K_* in gbfg.h).
enum KernelId { K_SAMPLE = 0, K_NOISE, K_DEPOSIT, K_SCAN, K_MEDIAN, K_PSD, K_INV_BLOCKS, K_SNR, K_AUX, K_COUNT };

// Brackets the launches issued during its lifetime with a pair of CUDA events on `st` when the
// calling thread has enabled profiling (gbfg_profile_enable); otherwise does nothing.
struct LaunchTimer {
    int slot;
    cudaStream_t st;
    LaunchTimer(int kernel_id, cudaStream_t stream);
    ~LaunchTimer();
};

#define GBFG_CUDA(call)                                                        \
    do {                                                                       \
        cudaError_t e__ = (call);                                              \
        if (e__ != cudaSuccess) return gbfg::set_cuda_error(e__, #call);       \
    } while (0)

#define GBFG_LAUNCH_CHECK(name)                                                \
    do {                                                                       \
        gbfg::count_launch();                                                  \
        cudaError_t e__ = cudaGetLastError();                                  \
        if (e__ != cudaSuccess) return gbfg::set_cuda_error(e__, name);        \
    } while (0)

// Programmatic dependent launch (sm_90+): the kernel is queued so that its CTAs may start while the kernel before
// it on the stream is still draining; it must call gbfg_wait_prior_kernel() before it touches anything that kernel
// wrote.  A kernel that lets its successor start early calls gbfg_let_next_kernel_start() (all its CTAs are
// resident by then, so the early CTAs of the successor can only take slots that are free).
template <typename... KArgs, typename... Args>
inline cudaError_t launch_dependent(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, Args... args)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr; cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kernel, KArgs(args)...);
}
#ifdef __CUDACC__
__device__ __forceinline__ void gbfg_wait_prior_kernel() { cudaGridDependencySynchronize(); }
__device__ __forceinline__ void gbfg_let_next_kernel_start() { cudaTriggerProgrammaticLaunchCompletion(); }
#endif

// Per-batch catalog table passed by value to kernels (<= GBFG_MAX_CAT catalogs).
struct CatTable {
    int32_t n_cat;
    int64_t offsets[GBFG_MAX_CAT + 1];
};

// Grid constants precomputed on the host (each a single IEEE operation, R2).
struct GridDev {
    double f_min, f_max, T, T2, halfT;
    int64_t n_bins;
    int32_t scale_log2;
};

inline GridDev make_grid_dev(const gbfg_grid *g)
{
    GridDev d;
    d.f_min = g->f_min; d.f_max = g->f_max; d.T = g->t_obs;
    d.T2 = g->t_obs * g->t_obs;
    d.halfT = 0.5 * g->t_obs;
    d.n_bins = g->n_bins; d.scale_log2 = g->scale_log2;
    return d;
}

// Dirty blocks.  The bins of a row are grouped in blocks of 2^dblk_log2 bins (>= 256, at most
// DIRTY_MAX_BLOCKS per row).  A subtraction stamps the blocks whose running-median OUTPUT can
// change: those within h bins of a bin it touched.  plan_kernel (median.cu) turns the stamps of
// one iteration into (a) the work list of the running median, (b) cum[c][b] = number of dirty
// blocks before block b, which lets the prefix of 1/S_n and the SNR test skip what did not change.
constexpr int DIRTY_MAX_BLOCKS = 16384;

inline int dirty_block_log2(int64_t n_bins)
{
    int L = 8;
    while (((n_bins + ((int64_t)1 << L) - 1) >> L) > DIRTY_MAX_BLOCKS) ++L;
    return L;
}
inline int dirty_blocks_per_row(int64_t n_bins)
{
    const int L = dirty_block_log2(n_bins);
    return (int)((n_bins + ((int64_t)1 << L) - 1) >> L);
}

struct DirtyView {
    const int *cum;     // [n_cat][n_dblk + 1], NULL: everything is dirty
    const int *range;   // [n_cat][2] first and last dirty block of each row (first > last: none)
    int n_dblk;
    int dblk_log2;
};

// Range-update deposit (deposit.cu): sources of at most DEP_NARROW bins add q with L2 atomics, wider
// ones write +q / -q into the difference array, scanned in tiles of DEP_SCAN_TILE bins.
constexpr int DEP_NARROW = 4;
constexpr int DEP_SCAN_TILE = 2048;

// Stamps written by a deposit / subtraction (deposit.cu): which scan tiles hold range updates, and
// which dirty blocks see a changed bin within h (blk_stamp NULL: not tracked).
struct DepositMarks {
    int *scan_stamp;    // [n_cat][scan_tiles]
    int scan_tiles;
    int *blk_stamp;     // [n_cat][n_dblk] or NULL
    int n_dblk;
    int dblk_log2;
    int med_h;          // half window
    int stamp;          // value written
    int64_t *live_sums; // nullable: [n_cat][scan_tiles], zero on entry: the sums of the difference array's tiles, kept by
                        // whoever writes a range update (the loop's test), so that the scan needs no pass of its own for them
};


// Stages (i) + (ii) in one kernel (sample.cu): where the drawn sources go
struct SampleDeposit {
    int64_t *spectrum;      // [n_cat][n_bins], accumulated into
    int64_t *diff;          // [n_cat][n_bins]
    int64_t *err_count;     // nullable
    int *wide_flag;
    DepositMarks mk;
    int64_t piece;          // > 0: catalogs are drawn in pieces of at most this many sources ...
    int (*after_piece)(void *ctx, int64_t i_begin, int64_t i_end);   // ... and this is called (host) after each launch
    void *ctx;
};

// What stage (iv) needs to subtract the sources it selects on the spot (snr.cu; spectrum NULL: it only selects)
struct SubtractView {
    int64_t *spectrum;      // [n_cat][n_bins]
    int64_t *diff;          // [n_cat][n_bins]
    int *wide_flag;
    DepositMarks mk;
    int scale_log2;
};

// Work list of the running median (median.cu): items[i] = (row, first output, outputs, 0).
struct MedianPlan {
    int4 *items;
    int *ctr;           // [0] number of items, [1] next item to take (both zero before plan_kernel)
    int4 *wide_items;   // [max_items] tiles left to the 64-bit-key kernel
    int *wide_ctr;      // [0] their number, [1] next to take
    int *cum;           // [n_cat][n_dblk + 1]
    int *range;         // [n_cat][2] first and last dirty block
    int n_dblk;
    int dblk_log2;
    int max_items;
    int *near_fold;     // SnrWork::any_near (nullable): plan_kernel folds word 1 into word 0
};

// What plan_kernel hands to the host before it clears the iteration's counters (loop.cu): n words of src copied to
// dst (mapped pinned host memory), then seq written at dst[flag_at].
struct PlanPublish {
    const int64_t *src;
    int64_t *dst;
    int n, flag_at;
    int64_t seq;
    int64_t *zero_sums;     // nullable: tile sums of the range updates after next (the other of two buffers), cleared here
    int zero_sums_n;
};

// A candidate record as the test reads it: one 32-byte sector, moved by one 256-bit access (four arrays cost four
// partly used sectors per record in the ordering pass, which scatters them)
struct __align__(32) CandRec {
    int64_t gk0;        // first bin (index into [n_cat][n_bins])
    double four_p;
    int64_t src;        // global source index
    int32_t w;          // width; 0 once resolved; negated once a test was near the threshold
    int32_t pad;
};

// Workspace of stage (iv) (snr.cu): the 128-bit fixed-point prefix of 1/psd and the candidate records.
struct SnrWork {
    void *pref;         // [n_cat][n_bins] 16-byte local prefixes
    void *tile_tot;     // [n_cat][pfx_tiles_per_row] 16-byte tile totals
    void *hdr;          // scale of the fixed point
    CandRec *cand_rec;  // [n_src_total] the records the test reads, one 32-byte sector each
    int64_t *cand_count;// [1 + n_cat]: number of records, per catalog
    // the records as first compacted (any order); cand_rec holds them ordered by (row, dirty
    // block of the first bin), which makes the gathers of the test coherent and lets it skip the
    // part of the list that lies outside the dirty range
    int64_t *tmp_gk0;   // [n_src_total]
    int32_t *tmp_w;
    double *tmp_4p;
    int64_t *tmp_src;
    int *bkt_count;     // [n_cat][n_dblk]      records per bucket, then the scatter cursor
    int *bkt_ext;       // [n_cat][n_dblk]      last block any record of the bucket reaches, then its prefix maximum
    int *bkt_reach;     // [n_cat][n_dblk]      first bucket with a record that reaches block b (n_dblk: none)
    int64_t *bkt_off;   // [n_cat][n_dblk + 1]  first record of each bucket (global record index)
    int *any_near;      // two ints.  [0]: a record was flagged near-threshold in an EARLIER pass (the whole list is tested
                        // from then on); read-only for the test, so that every CTA of one launch takes the same record
                        // range.  [1]: raised by the test of this pass; plan_kernel folds it into [0] between two passes
};

// ---------------------------------------------------------------------------------------------
// device helpers
// ---------------------------------------------------------------------------------------------

// catalog of global source index i (n_cat is small: linear scan for <= 4, else binary search)
__device__ __forceinline__ int cat_of(const CatTable &ct, int64_t i)
{
    if (ct.n_cat == 1) return 0;
    int lo = 0, hi = ct.n_cat;          // invariant: offsets[lo] <= i < offsets[hi]
    while (hi - lo > 1) {
        int mid = (lo + hi) >> 1;
        if (ct.offsets[mid] <= i) lo = mid; else hi = mid;
    }
    return lo;
}

// The integer triple and per-bin power of one source (R2).
struct SrcBins {
    int64_t k0, w_eff, q;
    double p;
    int status;     // 0 deposits, 1 DOMAIN, 2 RANGE
};

__device__ __forceinline__ SrcBins source_bins(const GridDev &g, double A, double f, double fdot)
{
    SrcBins s;
    s.k0 = 0; s.w_eff = 0; s.q = 0; s.p = 0.0; s.status = 1;
    if (!(A >= 0.0) || !(fdot >= 0.0) || !(f >= g.f_min) || !(f < g.f_max)) return s;
    double kk = floor((f - g.f_min) * g.T);
    if (!(kk < (double)g.n_bins)) return s;
    s.status = 2;
    double ww = ceil(fdot * g.T2);
    if (!(ww < 0x1p62)) return s;
    if (ww < 1.0) ww = 1.0;
    double P = (A * A) * g.halfT;
    double pp = P / ww;
    double qd = ldexp(pp, -g.scale_log2);
    if (!(qd < 0x1p62)) return s;
    s.k0 = (int64_t)kk;
    int64_t w = (int64_t)ww;
    int64_t room = g.n_bins - s.k0;
    s.w_eff = w < room ? w : room;
    s.p = pp;
    s.q = __double2ll_rn(qd);           // round half to even, as llrint
    s.status = 0;
    return s;
}

__device__ __forceinline__ void atomic_add_i64(int64_t *addr, int64_t v)
{
    atomicAdd(reinterpret_cast<unsigned long long *>(addr), (unsigned long long)v);
}

// One source into the spectrum of its row (stage ii; deposit.cu explains the two forms): v = +-q over
// [k0, k0 + w_eff).  spectrum / diff point to the row.  Also stamps the scan tiles and, when tracked, the dirty blocks.
__device__ __forceinline__ void deposit_one(const SrcBins &s, int64_t v, int64_t n_bins, int cat, int64_t *__restrict__ spectrum,
                                            int64_t *__restrict__ diff, int *__restrict__ wide_flag, const DepositMarks &mk)
{
    if (s.w_eff <= DEP_NARROW) {
        for (int64_t k = s.k0; k < s.k0 + s.w_eff; ++k) atomic_add_i64(spectrum + k, v);
    } else {
        atomic_add_i64(diff + s.k0, v);
        mk.scan_stamp[(int64_t)cat * mk.scan_tiles + s.k0 / DEP_SCAN_TILE] = mk.stamp;
        if (s.k0 + s.w_eff < n_bins) {
            atomic_add_i64(diff + s.k0 + s.w_eff, -v);
            mk.scan_stamp[(int64_t)cat * mk.scan_tiles + (s.k0 + s.w_eff) / DEP_SCAN_TILE] = mk.stamp;
        }
        *wide_flag = mk.stamp;
    }
    if (mk.blk_stamp) {
        // outputs k with |k - b| <= h see bin b (reflected ends included)
        int64_t lo = s.k0 - mk.med_h, hi = s.k0 + s.w_eff - 1 + mk.med_h;
        if (lo < 0) lo = 0;
        if (hi > n_bins - 1) hi = n_bins - 1;
        int *bs = mk.blk_stamp + (int64_t)cat * mk.n_dblk;
        for (int64_t b = lo >> mk.dblk_log2; b <= (hi >> mk.dblk_log2); ++b) bs[b] = mk.stamp;
    }
}

}  // namespace gbfg
