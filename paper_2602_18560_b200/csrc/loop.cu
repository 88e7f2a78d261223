// loop.cu — the C-ABI stage calls that need workspace, and stage (v): the subtraction loop of
// Appendix D steps 4-10 (R6), device resident, one small scalar
// read back per iteration.
//
// Shape of one gbfg_subtract_until_converged call:
//   prefix of 1/S_instr -> candidate records (pre-selection, R5)           once
//   per iteration:  running median + PSD of the tiles the last subtraction touched
//                   prefix of 1/S_n -> SNR test of the candidates -> counters to the host
//                   subtraction of the newly resolved (stamps the tiles it touches)
#include <string.h>

#include "gbfg_common.cuh"
#include <atomic>
#include <chrono>

namespace gbfg {

// from the other translation units
int scan_tiles_per_row(int64_t n_bins);
int launch_deposit(const GridDev &g, const CatTable &ct, const double *A, const double *f, const double *fdot,
                   const int64_t *sel_idx, const int64_t *sel_count, int64_t n_launch, int32_t sign,
                   int64_t *spectrum, int64_t *err_count, int64_t *diff, int64_t *tile_sums, int *wide_flag,
                   const DepositMarks &mk, cudaStream_t st, cudaEvent_t after_deposit = nullptr);
int launch_scan(int64_t n_bins, int n_cat, int64_t *spectrum, int64_t *diff, int64_t *tile_sums, int *wide_flag,
                const DepositMarks &mk, cudaStream_t st);
int median_max_items(int64_t n_bins);
int launch_plan(const int *blk_stamp, int stamp, bool all_dirty, int64_t n_bins, int n_cat, int window,
                const MedianPlan &pl, int64_t *zero_ptr, int zero_n, int64_t *out_count, unsigned long long *zero2_ptr,
                cudaStream_t st, const PlanPublish *pub = nullptr);
int launch_median(const int64_t *x, int64_t n_bins, int n_cat, int window, int64_t *med,
                  const double *s_instr, double *psd, double norm, int scale_log2,
                  const MedianPlan *plan, int4 *wide_items, int *wide_ctr, int *neg_flag,
                  unsigned long long *delta_bits, cudaStream_t st);
int launch_mean(const DirtyView *dv, const int64_t *x, int64_t n_bins, int n_cat, int window, int64_t *sum,
                const double *s_instr, double *psd, int scale_log2, int *neg_flag, unsigned long long *delta_bits,
                cudaStream_t st);
int pfx_tiles_per_row(int64_t n_bins);
size_t snr_pref_bytes(int64_t n_bins, int n_cat);
size_t snr_tile_off_bytes(int64_t n_bins, int n_cat);
size_t snr_hdr_bytes();
int launch_prefix_header(const double *arr, int64_t n, int64_t n_bins_row, const SnrWork &sw, cudaStream_t st);
int launch_inv_prefix(const double *psd, int64_t n_bins, int n_cat, const SnrWork &sw, const DirtyView &dv, cudaStream_t st);
int launch_cand_build(const GridDev &g, const CatTable &ct, const double *A, const double *f, const double *fdot,
                      const uint8_t *resolved, const double *s_instr, double rho_th, double *rho2_out,
                      const SnrWork &sw, cudaStream_t st);
int cand_build_begin(const CatTable &ct, int64_t n_bins, const SnrWork &sw, cudaStream_t st);
int cand_build_range(const GridDev &g, const CatTable &ct, const double *A, const double *f, const double *fdot,
                     const uint8_t *resolved, const double *s_instr, double rho_th, double *rho2_out,
                     const SnrWork &sw, int64_t i_begin, int64_t i_end, cudaStream_t st);
int cand_build_finish(const GridDev &g, const CatTable &ct, const SnrWork &sw, cudaStream_t st);
int launch_snr_cand(int64_t n_bins, int n_cat, const double *psd, double rho_th, uint8_t *resolved, double *rho2_out,
                    int64_t n_launch, int64_t *sel_idx, int64_t *sel_count, int64_t *near_count, int near_per_cat,
                    const int *abort_flag, bool use_prefix, const SnrWork &sw, const DirtyView &dv, int64_t *test_count,
                    const SubtractView *sub, const unsigned long long *delta_bits, double psd_rtol, cudaStream_t st);

// ------------------------------------------------------------------------------- workspace
constexpr int WS_COUNTERS = 7 * GBFG_MAX_CAT + 16;

// layout of `counters` (int64): what the host reads back each iteration comes first
//   [0 .. n_cat]            sel_count: total, per catalog
//   [1+n_cat .. 1+2 n_cat)  near-threshold counts per catalog
//   [1+2 n_cat]             flags word: bit 0 = a median was negative
//   [2+2 n_cat .. 3+3 n_cat) cand_count: total, per catalog
//   [3+3 n_cat .. 3+4 n_cat) running-median outputs computed, per catalog (accumulated over the call)
//   [3+4 n_cat .. 3+5 n_cat) SNR tests evaluated, per catalog (accumulated over the call)
//   [3+5 n_cat .. 3+6 n_cat) largest relative PSD change of this pass, per catalog, as binary64 bits (R13)
struct Workspace {
    int64_t *diff;        // [n_cat * n_bins]   difference array of the range-update deposit
    int64_t *tile_sums;   // [n_cat * scan_tiles]
    int64_t *live_sums[2]; // the same, kept by the loop's test itself: one buffer per parity of the iteration
    int *scan_stamp;      // [n_cat * scan_tiles]
    int *blk_stamp;       // [n_cat * n_dblk]        dirty-block stamps
    MedianPlan plan;      // work list of the running median, cum of the dirty blocks
    int64_t *sel_idx;     // [n_src_total]
    int64_t *counters;    // [WS_COUNTERS]
    int *wide_flag;
    SnrWork sw;
    size_t bytes;
};

static size_t align_up(size_t v) { return (v + 255) & ~(size_t)255; }

static Workspace carve(void *base, int64_t n_bins, int64_t n_src_total, int n_cat)
{
    Workspace w;
    size_t off = 0;
    char *b = (char *)base;
    const size_t nsrc = (size_t)(n_src_total > 0 ? n_src_total : 1);
    const size_t rows = (size_t)n_cat * (size_t)n_bins;
    auto take = [&](size_t bytes) { char *p = b + off; off += align_up(bytes); return p; };
    w.diff = (int64_t *)take(sizeof(int64_t) * rows);
    w.tile_sums = (int64_t *)take(sizeof(int64_t) * (size_t)n_cat * (size_t)scan_tiles_per_row(n_bins));
    w.scan_stamp = (int *)take(sizeof(int) * (size_t)n_cat * (size_t)scan_tiles_per_row(n_bins));
    const int n_dblk = dirty_blocks_per_row(n_bins);
    w.blk_stamp = (int *)take(sizeof(int) * (size_t)n_cat * (size_t)n_dblk);
    w.plan.n_dblk = n_dblk;
    w.plan.dblk_log2 = dirty_block_log2(n_bins);
    w.plan.max_items = n_cat * median_max_items(n_bins);
    w.plan.cum = (int *)take(sizeof(int) * (size_t)n_cat * (size_t)(n_dblk + 1));
    w.plan.range = (int *)take(sizeof(int) * 2 * (size_t)n_cat);
    w.plan.items = (int4 *)take(sizeof(int4) * (size_t)w.plan.max_items);
    w.plan.ctr = (int *)take(sizeof(int) * 4);
    w.plan.wide_items = (int4 *)take(sizeof(int4) * (size_t)w.plan.max_items);
    w.plan.wide_ctr = (int *)take(sizeof(int) * 4);
    w.sel_idx = (int64_t *)take(sizeof(int64_t) * nsrc);
    w.counters = (int64_t *)take(sizeof(int64_t) * WS_COUNTERS);
    w.wide_flag = (int *)take(sizeof(int) * (size_t)(1 + n_cat));   // flag, then one scan ticket per row
    w.sw.pref = take(snr_pref_bytes(n_bins, n_cat));
    w.sw.tile_tot = take(snr_tile_off_bytes(n_bins, n_cat));
    w.sw.hdr = take(snr_hdr_bytes());
    w.sw.cand_rec = (CandRec *)take(sizeof(CandRec) * nsrc);
    w.sw.cand_count = w.counters + 2 + 2 * n_cat;
    w.sw.tmp_gk0 = (int64_t *)take(sizeof(int64_t) * nsrc);
    w.sw.tmp_w = (int32_t *)take(sizeof(int32_t) * nsrc);
    w.sw.tmp_4p = (double *)take(sizeof(double) * nsrc);
    w.sw.tmp_src = (int64_t *)take(sizeof(int64_t) * nsrc);
    w.sw.bkt_count = (int *)take(sizeof(int) * (size_t)n_cat * (size_t)n_dblk);
    w.sw.bkt_ext = (int *)take(sizeof(int) * (size_t)n_cat * (size_t)n_dblk);
    w.sw.bkt_reach = (int *)take(sizeof(int) * (size_t)n_cat * (size_t)n_dblk);
    w.sw.bkt_off = (int64_t *)take(sizeof(int64_t) * (size_t)n_cat * (size_t)(n_dblk + 1));
    w.sw.any_near = (int *)take(2 * sizeof(int));
    w.plan.near_fold = w.sw.any_near;
    w.live_sums[0] = (int64_t *)take(sizeof(int64_t) * (size_t)n_cat * (size_t)scan_tiles_per_row(n_bins));
    w.live_sums[1] = (int64_t *)take(sizeof(int64_t) * (size_t)n_cat * (size_t)scan_tiles_per_row(n_bins));
    w.bytes = off;
    return w;
}

static int make_cat_table(const int64_t *offsets, int n_cat, CatTable *ct)
{
    if (!offsets || n_cat < 1) return GBFG_ERR_INVALID_ARG;
    if (n_cat > GBFG_MAX_CAT) return GBFG_ERR_UNSUPPORTED;
    if (offsets[0] != 0) return GBFG_ERR_INVALID_ARG;
    ct->n_cat = n_cat;
    for (int c = 0; c <= n_cat; ++c) {
        if (c && offsets[c] < offsets[c - 1]) return GBFG_ERR_INVALID_ARG;
        ct->offsets[c] = offsets[c];
    }
    for (int c = n_cat + 1; c <= GBFG_MAX_CAT; ++c) ct->offsets[c] = offsets[n_cat];
    return GBFG_OK;
}

static int valid_grid(const gbfg_grid *g)
{
    return g && g->struct_size == sizeof(gbfg_grid) && g->n_bins >= 1 && g->n_bins < 2147483648ll &&
           g->f_min > 0.0 && g->f_max > g->f_min && g->t_obs > 0.0 && g->scale_log2 >= -1000 && g->scale_log2 <= 0;
}

// pinned host scratch for the per-iteration readback (one per host thread), mapped: the plan kernel stores the
// iteration's counters into it, then a sequence number in its last word
constexpr int HOST_SEQ_AT = WS_COUNTERS - 1;
static int64_t *host_scratch()
{
    static thread_local int64_t *p = nullptr;
    if (!p) {
        if (cudaHostAlloc((void **)&p, sizeof(int64_t) * WS_COUNTERS, cudaHostAllocPortable | cudaHostAllocMapped) != cudaSuccess) {
            (void)cudaGetLastError();
            p = nullptr;
        } else {
            memset(p, 0, sizeof(int64_t) * WS_COUNTERS);
        }
    }
    return p;
}

// the host's wait for the counters of one iteration: the sequence number the plan kernel writes behind them.
// ev_plan (recorded behind that kernel) is looked at now and then, so that a failed launch ends the wait.
static int wait_published(const int64_t *host, int64_t seq, cudaEvent_t ev_plan)
{
    const volatile int64_t *flag = host + HOST_SEQ_AT;
    for (unsigned spins = 1;; ++spins) {
        if (*flag == seq) break;
        if ((spins & 2047u) == 0u) {
            const cudaError_t e = cudaEventQuery(ev_plan);
            if (e == cudaSuccess) {
                if (*flag == seq) break;
                return set_cuda_error(cudaErrorUnknown, "plan_kernel did not publish the counters");
            }
            if (e != cudaErrorNotReady) return set_cuda_error(e, "plan_kernel");
        }
    }
    std::atomic_thread_fence(std::memory_order_acquire);
    return GBFG_OK;
}

// device arena and stream of gbfg_simulate_host, one per host thread
struct HostCallCache { char *base; size_t bytes; int device; cudaStream_t stream; };
static HostCallCache &host_call_cache()
{
    static thread_local HostCallCache c = {nullptr, 0, -1, nullptr};
    return c;
}

// event that marks the per-iteration readback (one per host thread)
static thread_local cudaEvent_t g_ev_read = nullptr;
static cudaEvent_t readback_event()
{
    cudaEvent_t &ev = g_ev_read;
    if (!ev && cudaEventCreateWithFlags(&ev, cudaEventDisableTiming) != cudaSuccess) { (void)cudaGetLastError(); ev = nullptr; }
    return ev;
}

// side stream on which the plan of the next pass runs next to the scan of the subtraction (one per host thread)
struct SideStream { cudaStream_t s; cudaEvent_t ev_plan, ev_aux, ev_noise; cudaStream_t copy; cudaEvent_t ev_copy; };
static SideStream &side_stream_slot()
{
    static thread_local SideStream ss = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};
    return ss;
}
static SideStream *side_stream_if_any() { return side_stream_slot().s ? &side_stream_slot() : nullptr; }
static SideStream *side_stream()
{
    SideStream &ss = side_stream_slot();
    if (!ss.s) {
        if (cudaStreamCreateWithFlags(&ss.s, cudaStreamNonBlocking) != cudaSuccess ||
            cudaEventCreateWithFlags(&ss.ev_plan, cudaEventDisableTiming) != cudaSuccess ||
            cudaEventCreateWithFlags(&ss.ev_aux, cudaEventDisableTiming) != cudaSuccess ||
            cudaEventCreateWithFlags(&ss.ev_noise, cudaEventDisableTiming) != cudaSuccess ||
            cudaStreamCreateWithFlags(&ss.copy, cudaStreamNonBlocking) != cudaSuccess ||
            cudaEventCreateWithFlags(&ss.ev_copy, cudaEventDisableTiming) != cudaSuccess) {
            (void)cudaGetLastError();
            ss.s = nullptr;
            return nullptr;
        }
    }
    return &ss;
}

// gbfg_simulate_host: the PSD starts its way to the (pinned) host buffer while the loop still runs.  Once a pass
// recomputes less than a tenth of the outputs, the PSD as it stands goes out on a copy stream; a block of 2^dblk_log2 bins
// that a later subtraction makes dirty carries a later stamp (deposit.cu), and exactly those blocks are stored again at
// the end by psd_patch_kernel, straight into the mapped host buffer.  Never changes a result: every bin of the host
// buffer is written last with its final value.
struct EarlyOut {
    double *host_psd;        // destination of the copy (pinned host memory) ...
    double *host_psd_dev;    // ... and the address kernels store to it through
    size_t bytes;
    cudaStream_t copy_stream;   // the copy and every patch run on this stream, in this order
    int started_after;       // iteration after which the PSD began to go out (-1: it did not)
    int patched_upto;        // blocks stamped up to this iteration have been stored again since
    size_t psd_sent;         // bytes of the PSD copied so far: it leaves in pieces, one per iteration (loop_body)
    double t_last;           // host clock [s] when the last iteration's counters were seen (0: not yet)
    // the resolved flags: final once the last test of a loop that runs to its cap is done, so their copy can run next
    // to the closing estimator pass
    uint8_t *host_resolved;  // nullable
    size_t resolved_bytes;
    cudaEvent_t ev_last_test;
    bool resolved_out;       // the copy of the final flags is queued on copy_stream
};
constexpr int EARLY_PATCH_EVERY = 4;       // iterations between two patches while the loop runs

// blocks with after < stamp <= upto, straight into the host buffer.  Runs next to the loop's kernels: a block that is
// stamped again meanwhile (whatever stamp this kernel then sees) is covered by a later patch, since stamps only grow.
__global__ void __launch_bounds__(256)
psd_patch_kernel(const double *__restrict__ psd, double *__restrict__ host_psd, const int *__restrict__ blk_stamp,
                 int n_dblk, int dblk_log2, int64_t n_bins, int after, int upto)
{
    const int64_t row = blockIdx.y;
    for (int b = blockIdx.x; b < n_dblk; b += gridDim.x) {
        const int stamp = ((const volatile int *)blk_stamp)[row * n_dblk + b];
        if (stamp <= after || stamp > upto) continue;
        const int64_t k0 = (int64_t)b << dblk_log2;
        int64_t k1 = k0 + ((int64_t)1 << dblk_log2);
        if (k1 > n_bins) k1 = n_bins;
        for (int64_t k = k0 + threadIdx.x; k < k1; k += blockDim.x) host_psd[row * n_bins + k] = psd[row * n_bins + k];
    }
}

static int launch_psd_patch(const EarlyOut &eo, const double *dev_psd, const int *blk_stamp, int n_dblk, int dblk_log2,
                            int64_t n_bins, int n_cat, int after, int upto)
{
    const int gx = n_dblk < 4 * sm_count() ? n_dblk : 4 * sm_count();
    psd_patch_kernel<<<dim3((unsigned)gx, (unsigned)n_cat), 256, 0, eo.copy_stream>>>(dev_psd, eo.host_psd_dev, blk_stamp, n_dblk,
                                                                                       dblk_log2, n_bins, after, upto);
    GBFG_LAUNCH_CHECK("psd_patch_kernel");
    return GBFG_OK;
}

// Everything above that is kept per host thread (stream, events, device arena) belongs to the device that was current
// when it was made.  A thread that comes back with another current device gets fresh ones (a stream or an event of one
// device is an invalid handle under another; the mapped host scratch is portable and stays).
static void release_thread_resources()
{
    HostCallCache &cc = host_call_cache();
    if (cc.stream) { cudaStreamSynchronize(cc.stream); cudaStreamDestroy(cc.stream); cc.stream = nullptr; }
    if (cc.base) { cudaFree(cc.base); cc.base = nullptr; cc.bytes = 0; }
    SideStream *side = side_stream_if_any();
    if (side) {                                          // the loop's side stream and its events
        cudaStreamSynchronize(side->s);
        cudaEventDestroy(side->ev_plan);
        cudaEventDestroy(side->ev_aux);
        cudaEventDestroy(side->ev_noise);
        if (side->copy) { cudaStreamSynchronize(side->copy); cudaStreamDestroy(side->copy); side->copy = nullptr; }
        if (side->ev_copy) { cudaEventDestroy(side->ev_copy); side->ev_copy = nullptr; }
        cudaStreamDestroy(side->s);
        side->s = nullptr;
    }
    if (g_ev_read) { cudaEventDestroy(g_ev_read); g_ev_read = nullptr; }
    (void)cudaGetLastError();
}

static int bind_thread_to_current_device()
{
    static thread_local int tl_dev = -1;
    int dev = 0;
    GBFG_CUDA(cudaGetDevice(&dev));
    if (tl_dev != dev) {
        if (tl_dev >= 0) {
            // the old resources are destroyed with their own device current
            if (cudaSetDevice(tl_dev) == cudaSuccess) release_thread_resources();
            (void)cudaGetLastError();
            GBFG_CUDA(cudaSetDevice(dev));
        }
        tl_dev = dev;
    }
    return GBFG_OK;
}

// an error return leaves nothing of the call in flight: kernels queued on the side stream still use the caller's buffers
static int drain_on_error(int rc, cudaStream_t st)
{
    if (rc != GBFG_OK) {
        SideStream *side = side_stream_if_any();
        if (side) (void)cudaStreamSynchronize(side->s);
        (void)cudaStreamSynchronize(st);
        (void)cudaGetLastError();
    }
    return rc;
}

static DepositMarks plain_marks(const Workspace &w, int64_t n_bins, int stamp)
{
    DepositMarks mk;
    mk.scan_stamp = w.scan_stamp; mk.scan_tiles = scan_tiles_per_row(n_bins);
    mk.blk_stamp = nullptr; mk.n_dblk = 0; mk.dblk_log2 = 0; mk.med_h = 0;
    mk.stamp = stamp;
    mk.live_sums = nullptr;
    return mk;
}

}  // namespace gbfg

using namespace gbfg;

extern "C" size_t gbfg_workspace_bytes(const gbfg_grid *grid, int64_t n_src_total, int32_t n_cat)
{
    if (!valid_grid(grid) || n_cat < 1 || n_cat > GBFG_MAX_CAT || n_src_total < 0) return 0;
    return carve(nullptr, grid->n_bins, n_src_total, n_cat).bytes;
}

extern "C" int gbfg_deposit(const gbfg_grid *grid, const double *dev_A, const double *dev_f, const double *dev_fdot,
                            const int64_t *offsets, int32_t n_cat,
                            const int64_t *dev_sel_idx, const int64_t *dev_sel_count, int32_t sign,
                            int64_t *dev_spectrum, int64_t *dev_err_count,
                            void *workspace, size_t workspace_bytes, void *stream)
{
    if (!valid_grid(grid) || !dev_spectrum || (sign != 1 && sign != -1)) return GBFG_ERR_INVALID_ARG;
    if ((dev_sel_idx == nullptr) != (dev_sel_count == nullptr)) return GBFG_ERR_INVALID_ARG;
    CatTable ct;
    int rc = make_cat_table(offsets, n_cat, &ct);
    if (rc) return rc;
    const int64_t n = ct.offsets[n_cat];
    if (n > 0 && (!dev_A || !dev_f || !dev_fdot)) return GBFG_ERR_INVALID_ARG;
    if (!workspace || ((uintptr_t)workspace & 31u)) return GBFG_ERR_WORKSPACE;     // (256-bit accesses to its records)
    Workspace w = carve(workspace, grid->n_bins, n, n_cat);
    if (workspace_bytes < w.bytes) return GBFG_ERR_WORKSPACE;
    rc = check_device();
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    GBFG_CUDA(cudaMemsetAsync(w.diff, 0, sizeof(int64_t) * (size_t)n_cat * (size_t)grid->n_bins, st));
    GBFG_CUDA(cudaMemsetAsync(w.wide_flag, 0, sizeof(int) * (size_t)(1 + n_cat), st));
    GBFG_CUDA(cudaMemsetAsync(w.scan_stamp, 0, sizeof(int) * (size_t)n_cat * (size_t)scan_tiles_per_row(grid->n_bins), st));
    return launch_deposit(make_grid_dev(grid), ct, dev_A, dev_f, dev_fdot, dev_sel_idx, dev_sel_count, n, sign,
                          dev_spectrum, dev_err_count, w.diff, w.tile_sums, w.wide_flag,
                          plain_marks(w, grid->n_bins, 1), st);
}

extern "C" int gbfg_snr_select(const gbfg_grid *grid, const double *dev_A, const double *dev_f, const double *dev_fdot,
                               const int64_t *offsets, int32_t n_cat, const double *dev_psd, double rho_th,
                               uint8_t *dev_resolved, double *dev_rho2_out,
                               int64_t *dev_sel_idx, int64_t *dev_sel_count, int64_t *dev_near_count,
                               void *workspace, size_t workspace_bytes, void *stream)
{
    if (!valid_grid(grid) || !dev_psd || !dev_resolved || !dev_sel_idx || !dev_sel_count) return GBFG_ERR_INVALID_ARG;
    if (!(rho_th >= 0.0)) return GBFG_ERR_INVALID_ARG;
    CatTable ct;
    int rc = make_cat_table(offsets, n_cat, &ct);
    if (rc) return rc;
    const int64_t n = ct.offsets[n_cat];
    if (n > 0 && (!dev_A || !dev_f || !dev_fdot)) return GBFG_ERR_INVALID_ARG;
    if (!workspace || ((uintptr_t)workspace & 31u)) return GBFG_ERR_WORKSPACE;     // (256-bit accesses to its records)
    Workspace w = carve(workspace, grid->n_bins, n, n_cat);
    if (workspace_bytes < w.bytes) return GBFG_ERR_WORKSPACE;
    rc = check_device();
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    const GridDev g = make_grid_dev(grid);
    GBFG_CUDA(cudaMemsetAsync(dev_sel_count, 0, sizeof(int64_t) * (size_t)(1 + n_cat), st));
    GBFG_CUDA(cudaMemsetAsync(w.sw.cand_count, 0, sizeof(int64_t) * (size_t)(1 + n_cat), st));
    if (n <= 0) return GBFG_OK;
    // every unresolved valid source is a candidate (no pre-selection: the PSD is the caller's)
    rc = launch_prefix_header(dev_psd, (int64_t)n_cat * grid->n_bins, grid->n_bins, w.sw, st);
    if (rc) return rc;
    const DirtyView all_dirty = {nullptr, nullptr, 0, 0};
    rc = launch_inv_prefix(dev_psd, grid->n_bins, n_cat, w.sw, all_dirty, st);
    if (rc) return rc;
    rc = launch_cand_build(g, ct, dev_A, dev_f, dev_fdot, dev_resolved, nullptr, rho_th, dev_rho2_out, w.sw, st);
    if (rc) return rc;
    return launch_snr_cand(grid->n_bins, n_cat, dev_psd, rho_th, dev_resolved, dev_rho2_out, n, dev_sel_idx,
                           dev_sel_count, dev_near_count, 0, nullptr, true, w.sw, all_dirty, nullptr, nullptr, nullptr, 0.0, st);
}

// workspace state the loop starts from (also what a deposit needs: zero difference array and stamps)
static int loop_init_workspace(const Workspace &w, int64_t nb, int n_cat, cudaStream_t st)
{
    const size_t row_bytes = sizeof(int64_t) * (size_t)n_cat * (size_t)nb;
    GBFG_CUDA(cudaMemsetAsync(w.diff, 0, row_bytes, st));
    GBFG_CUDA(cudaMemsetAsync(w.wide_flag, 0, sizeof(int) * (size_t)(1 + n_cat), st));
    GBFG_CUDA(cudaMemsetAsync(w.counters, 0, sizeof(int64_t) * WS_COUNTERS, st));
    GBFG_CUDA(cudaMemsetAsync(w.scan_stamp, 0, sizeof(int) * (size_t)n_cat * (size_t)scan_tiles_per_row(nb), st));
    GBFG_CUDA(cudaMemsetAsync(w.live_sums[0], 0, 2 * align_up(sizeof(int64_t) * (size_t)n_cat * (size_t)scan_tiles_per_row(nb)), st));
    GBFG_CUDA(cudaMemsetAsync(w.blk_stamp, 0, sizeof(int) * (size_t)n_cat * (size_t)w.plan.n_dblk, st));
    return GBFG_OK;
}

// candidate records: with pre-selection, only sources whose rho^2 against S_instr reaches the threshold.
// First half: the header and (for the pre-selection) the prefix of 1/S_instr, which need nothing of the catalog.
static int loop_prefix_s_instr(const GridDev &g, const double *dev_s_instr, bool preselect, const Workspace &w, cudaStream_t st)
{
    const DirtyView all_dirty = {nullptr, nullptr, 0, 0};
    int rc = launch_prefix_header(dev_s_instr, g.n_bins, g.n_bins, w.sw, st);
    if (rc) return rc;
    if (preselect) rc = launch_inv_prefix(dev_s_instr, g.n_bins, 1, w.sw, all_dirty, st);
    return rc;
}

static int loop_build_candidates(const GridDev &g, const CatTable &ct, const double *dev_A, const double *dev_f,
                                 const double *dev_fdot, const uint8_t *dev_resolved, const double *dev_s_instr,
                                 double rho_th, bool preselect, const Workspace &w, cudaStream_t st)
{
    return launch_cand_build(g, ct, dev_A, dev_f, dev_fdot, dev_resolved, preselect ? dev_s_instr : nullptr, rho_th, nullptr,
                             w.sw, st);
}

static int loop_validate(const gbfg_grid *grid, const gbfg_iter_params *params)
{
    if (!valid_grid(grid) || !params || params->struct_size != sizeof(gbfg_iter_params)) return GBFG_ERR_INVALID_ARG;
    const int W = params->window;
    const bool use_mean = (params->flags & GBFG_FLAG_ESTIMATOR_MEAN) != 0;
    if (W < 1 || (W & 1) == 0 || params->max_iter < 1 || !(params->rho_th >= 0.0) || (!use_mean && !(params->median_norm > 0.0)))
        return GBFG_ERR_INVALID_ARG;
    if (W > GBFG_MAX_WINDOW) return GBFG_ERR_UNSUPPORTED;
    if (grid->n_bins < W / 2 + 1) return GBFG_ERR_INVALID_ARG;
    return GBFG_OK;
}

// the loop proper.  prepared: the caller has initialised the workspace and built the candidate records (gbfg_simulate
// does both next to the deposit).
static int loop_body(const gbfg_grid *grid, const double *dev_A, const double *dev_f,
                     const double *dev_fdot, const int64_t *offsets, int32_t n_cat,
                     const double *dev_s_instr, const gbfg_iter_params *params,
                     int64_t *dev_spectrum, int64_t *dev_median, double *dev_psd,
                     uint8_t *dev_resolved, gbfg_iter_result *host_results,
                     void *workspace, size_t workspace_bytes, void *stream, bool prepared,
                     cudaEvent_t records_ready, EarlyOut *eo = nullptr)
{
    int rc = loop_validate(grid, params);
    if (rc) return rc;
    if (!dev_s_instr || !dev_spectrum || !dev_median || !dev_psd || !dev_resolved || !host_results) return GBFG_ERR_INVALID_ARG;
    const int W = params->window;
    const bool use_mean = (params->flags & GBFG_FLAG_ESTIMATOR_MEAN) != 0;
    CatTable ct;
    rc = make_cat_table(offsets, n_cat, &ct);
    if (rc) return rc;
    const int64_t n = ct.offsets[n_cat];
    if (n > 0 && (!dev_A || !dev_f || !dev_fdot)) return GBFG_ERR_INVALID_ARG;
    if (!workspace || ((uintptr_t)workspace & 31u)) return GBFG_ERR_WORKSPACE;     // (256-bit accesses to its records)
    Workspace w = carve(workspace, grid->n_bins, n, n_cat);
    if (workspace_bytes < w.bytes) return GBFG_ERR_WORKSPACE;
    rc = check_device();
    if (rc) return rc;
    int64_t *host = host_scratch();
    if (!host) return set_cuda_error(cudaErrorMemoryAllocation, "cudaHostAlloc");
    cudaStream_t st = (cudaStream_t)stream;
    const GridDev g = make_grid_dev(grid);
    const int64_t nb = grid->n_bins;

    int64_t *sel_count = w.counters;                    // [1 + n_cat]
    int64_t *near = w.counters + 1 + n_cat;             // [n_cat]
    int *neg_flag = (int *)(w.counters + 1 + 2 * n_cat);
    const size_t n_iter_counters = (size_t)(1 + 2 * n_cat);      // zeroed every iteration
    const size_t n_read_all = (size_t)(3 + 6 * n_cat);           // ... + flags + cand_count + work counters + PSD change
    const double psd_rtol = params->psd_rtol > 0.0 ? params->psd_rtol : 0.0;
    unsigned long long *delta_all = (unsigned long long *)(w.counters + 3 + 5 * n_cat);
    const int i_delta = 3 + 5 * n_cat;
    int64_t *med_outputs = w.counters + 3 + 3 * n_cat, *snr_tests = w.counters + 3 + 4 * n_cat;
    const int i_med = 3 + 3 * n_cat, i_tests = 3 + 4 * n_cat;
    const int i_flags = 1 + 2 * n_cat, i_cand = 2 + 2 * n_cat;
    bool preselect = (params->flags & GBFG_FLAG_NO_PRESELECT) == 0;
    const bool incremental = (params->flags & GBFG_FLAG_NO_INCREMENTAL) == 0;

    const DirtyView all_dirty = {nullptr, nullptr, 0, 0};
    const DirtyView dirty = {w.plan.cum, w.plan.range, w.plan.n_dblk, w.plan.dblk_log2};
    if (!prepared) {
        rc = loop_init_workspace(w, nb, n_cat, st);
        if (rc) return rc;
        rc = loop_prefix_s_instr(g, dev_s_instr, preselect, w, st);
        if (rc) return rc;
        rc = loop_build_candidates(g, ct, dev_A, dev_f, dev_fdot, dev_resolved, dev_s_instr, params->rho_th, preselect, w, st);
        if (rc) return rc;
    }

    bool done[GBFG_MAX_CAT];
    for (int c = 0; c < n_cat; ++c) {
        memset(&host_results[c], 0, sizeof(gbfg_iter_result));
        done[c] = false;
    }
    int64_t n_cand = n;                                 // upper bound until the first readback
    bool plan_queued = false;
    SideStream *side = side_stream();
    if (!side) return set_cuda_error(cudaErrorMemoryAllocation, "side stream");
    cudaEvent_t ev_read = readback_event();
    if (!ev_read) return set_cuda_error(cudaErrorMemoryAllocation, "cudaEventCreate");
    int n_done = 0;
    int64_t med_outputs_seen = 0;
    for (int it = 0; it < params->max_iter && n_done < n_cat; ++it) {
        // what the last subtraction made dirty (everything, the first time): work list + cum
        if (plan_queued) {
            GBFG_CUDA(cudaStreamWaitEvent(st, side->ev_plan, 0));
        } else {
            rc = launch_plan(w.blk_stamp, it, it == 0 || !incremental, nb, n_cat, W, w.plan, w.counters, (int)n_iter_counters,
                             med_outputs, delta_all, st);
            if (rc) return rc;
        }
        plan_queued = false;
        // second stop rule (R13): from the second pass on the estimator also records the largest relative PSD change
        unsigned long long *delta = (psd_rtol > 0.0 && it > 0) ? delta_all : nullptr;
        if (use_mean) {      // eq. (D1): HBM bound; tiles without a dirty block keep their sums and PSD
            rc = launch_mean(&dirty, dev_spectrum, nb, n_cat, W, dev_median, dev_s_instr, dev_psd, grid->scale_log2, neg_flag, delta, st);
        } else {
            rc = launch_median(dev_spectrum, nb, n_cat, W, dev_median, dev_s_instr, dev_psd, params->median_norm,
                               grid->scale_log2, &w.plan, nullptr, nullptr, neg_flag, delta, st);
        }
        if (rc) return rc;
        // gbfg_simulate builds the candidate records on the side stream; the first estimator pass above does not need
        // them, the prefix below reuses the buffers their pre-selection reads (the prefix of 1/S_instr)
        if (it == 0 && records_ready) GBFG_CUDA(cudaStreamWaitEvent(st, records_ready, 0));
        rc = launch_inv_prefix(dev_psd, nb, n_cat, w.sw, dirty, st);
        if (rc) return rc;
        // The test subtracts what it selects on the spot (stage v, eq. D4) and stamps the blocks that become dirty.
        DepositMarks mk = plain_marks(w, nb, it + 1);
        mk.blk_stamp = w.blk_stamp; mk.n_dblk = w.plan.n_dblk; mk.dblk_log2 = w.plan.dblk_log2; mk.med_h = W / 2;
        // the test keeps the sums of the range updates' tiles itself (two buffers: the plan behind this iteration's test
        // clears the one the next test will add into, which the scan before last was the last to read)
        mk.live_sums = w.live_sums[it & 1];
        const SubtractView sub = {dev_spectrum, w.diff, w.wide_flag, mk, grid->scale_log2};
        rc = launch_snr_cand(nb, n_cat, dev_psd, params->rho_th, dev_resolved, nullptr, n_cand, w.sel_idx, sel_count,
                             near, 1, preselect ? neg_flag : nullptr, true, w.sw, dirty, snr_tests, &sub, delta, psd_rtol, st);
        if (rc) return rc;
        if (eo && eo->host_resolved && eo->resolved_bytes && it + 1 == params->max_iter) {
            GBFG_CUDA(cudaEventRecord(eo->ev_last_test, st));
            GBFG_CUDA(cudaStreamWaitEvent(eo->copy_stream, eo->ev_last_test, 0));
            GBFG_CUDA(cudaMemcpyAsync(eo->host_resolved, dev_resolved, eo->resolved_bytes, cudaMemcpyDeviceToHost, eo->copy_stream));
            eo->resolved_out = true;
        }
        GBFG_CUDA(cudaEventRecord(ev_read, st));            // the test is queued; its counters reach the host through the plan below
        // Everything below is queued before the host has seen the counters (a pass that selected nothing makes
        // it a no-op), so the GPU does not idle while the host waits for the scalar that decides whether the
        // loop goes on: the scan of the wide sources' range updates into the spectrum ...
        rc = launch_scan(nb, n_cat, dev_spectrum, w.diff, w.tile_sums, w.wide_flag, mk, st);
        if (rc) return rc;
        // ... and, on the side stream next to it, the plan of the next pass: it stores the test's counters into the
        // host's mapped scratch (no copy engine between the test and the scan), clears them and reads the stamps
        // the test wrote.  After the last iteration it is the plan of the closing median pass.
        {
            const bool closing = it + 1 == params->max_iter;
            static thread_local int64_t seq_counter = 0;
            const PlanPublish pub = {w.counters, host, (int)n_read_all, HOST_SEQ_AT, ++seq_counter, w.live_sums[(it + 1) & 1],
                                     n_cat * scan_tiles_per_row(nb)};
            GBFG_CUDA(cudaStreamWaitEvent(side->s, ev_read, 0));
            rc = launch_plan(w.blk_stamp, it + 1, !incremental, nb, n_cat, W, w.plan, closing ? nullptr : w.counters,
                             closing ? 0 : (int)n_iter_counters, med_outputs,
                             closing ? nullptr : delta_all, side->s, &pub);
            if (rc) return rc;
            GBFG_CUDA(cudaEventRecord(side->ev_plan, side->s));
            plan_queued = true;
            rc = wait_published(host, pub.seq, side->ev_plan);
            if (rc) return rc;
        }
        if (preselect && host[i_flags] != 0) {
            if (plan_queued) { GBFG_CUDA(cudaStreamWaitEvent(st, side->ev_plan, 0)); plan_queued = false; }   // it saw no stamps: made again
            // A negative median: S_n >= S_instr no longer holds, so the pre-selection is not valid
            // (the caller's spectrum does not contain the catalog).  Every unresolved source becomes
            // a candidate, and this iteration's test, which did nothing (as did the scan queued behind it),
            // is run on them.
            preselect = false;
            if (eo) eo->resolved_out = false;            // the test runs again: the flags go out at the end
            GBFG_CUDA(cudaMemsetAsync(w.sw.cand_count, 0, sizeof(int64_t) * (size_t)(1 + n_cat), st));
            rc = launch_cand_build(g, ct, dev_A, dev_f, dev_fdot, dev_resolved, nullptr, params->rho_th, nullptr, w.sw, st);
            if (rc) return rc;
            rc = launch_snr_cand(nb, n_cat, dev_psd, params->rho_th, dev_resolved, nullptr, n, w.sel_idx, sel_count,
                                 near, 1, nullptr, true, w.sw, all_dirty, snr_tests, &sub, delta, psd_rtol, st);
            if (rc) return rc;
            GBFG_CUDA(cudaMemcpyAsync(host, w.counters, sizeof(int64_t) * n_read_all, cudaMemcpyDeviceToHost, st));
            rc = launch_scan(nb, n_cat, dev_spectrum, w.diff, w.tile_sums, w.wide_flag, mk, st);
            if (rc) return rc;
            GBFG_CUDA(cudaStreamSynchronize(st));
            for (int c = 0; c < n_cat; ++c) host_results[c].n_candidates = 0;
        }
        n_cand = host[i_cand];
        const int64_t total = host[0];
        {   // outputs the estimator recomputed in this pass (the plan accumulates them, loop.cu's counter layout)
            int64_t outs = 0;
            for (int c = 0; c < n_cat; ++c) outs += host[i_med + c];
            const int64_t last_pass = outs - med_outputs_seen;
            med_outputs_seen = outs;
            if (eo && incremental && !use_mean) {
                const double t_now = std::chrono::duration<double>(std::chrono::steady_clock::now().time_since_epoch()).count();
                if (eo->started_after < 0) {
                    if (it >= 1 && last_pass * 10 < (int64_t)n_cat * nb) {
                        eo->started_after = eo->patched_upto = it;
                        eo->psd_sent = 0;
                    }
                }
                if (eo->started_after >= 0 && eo->psd_sent < eo->bytes) {
                    // The PSD leaves in pieces, one per iteration, each sized to be through the link before the next plan
                    // kernel hands over its counters: 30 MB in one copy kept the link busy for half a millisecond, and
                    // the few stores and the system fence of every plan in that time queued up behind it while the host
                    // (and with it the next pass) waited for them: the loop took 0.45 ms longer than without the copy.
                    const double dt = eo->t_last > 0.0 ? t_now - eo->t_last : 50e-6;
                    double want = 0.7 * dt * 50e9;                       // bytes at 50 GB/s in 70 % of the last iteration's time
                    if (want < 1048576.0) want = 1048576.0;
                    if (want > 8388608.0) want = 8388608.0;
                    size_t sz = (size_t)want & ~(size_t)4095;
                    if (sz > eo->bytes - eo->psd_sent) sz = eo->bytes - eo->psd_sent;
                    GBFG_CUDA(cudaMemcpyAsync((char *)eo->host_psd + eo->psd_sent, (const char *)dev_psd + eo->psd_sent, sz,
                                              cudaMemcpyDeviceToHost, eo->copy_stream));
                    eo->psd_sent += sz;
                }
                eo->t_last = t_now;
                if (eo->started_after >= 0 && it - eo->patched_upto >= EARLY_PATCH_EVERY) {
                    // the estimator passes up to `it` are done: blocks stamped in (patched_upto, it] hold what they will
                    // keep unless a later subtraction stamps them again
                    rc = launch_psd_patch(*eo, dev_psd, w.blk_stamp, w.plan.n_dblk, w.plan.dblk_log2, nb, n_cat, eo->patched_upto, it);
                    if (rc) return rc;
                    eo->patched_upto = it;
                }
            }
        }
        for (int c = 0; c < n_cat; ++c) {
            gbfg_iter_result &r = host_results[c];
            if (r.n_candidates == 0) r.n_candidates = n_cat == 1 ? host[i_cand] : host[i_cand + 1 + c];
            if (done[c]) continue;
            if (delta) {                                 // S_n converged: the test of this pass did not run for this catalog
                double d;
                memcpy(&d, &host[i_delta + c], sizeof(double));
                if (d <= psd_rtol) {
                    if (it < GBFG_MAX_ITER_TRACE) r.n_new_per_iter[it] = 0;
                    done[c] = true; ++n_done; r.n_iter = it + 1; r.converged = 2;
                    continue;
                }
            }
            const int64_t n_new = host[1 + c];
            if (it < GBFG_MAX_ITER_TRACE) r.n_new_per_iter[it] = n_new;
            r.n_resolved += n_new;
            r.n_near_threshold += host[1 + n_cat + c];
            if (n_new == 0) { done[c] = true; ++n_done; r.n_iter = it + 1; r.converged = 1; }
        }
        if (total == 0) break;
    }
    if (n_done < n_cat) {
        // cap hit: the PSD must match the returned residual (rows of converged catalogs are unchanged)
        for (int c = 0; c < n_cat; ++c)
            if (!done[c]) { host_results[c].n_iter = params->max_iter; host_results[c].converged = 0; }
        if (plan_queued) {
            GBFG_CUDA(cudaStreamWaitEvent(st, side->ev_plan, 0));
        } else {
            rc = launch_plan(w.blk_stamp, params->max_iter, !incremental, nb, n_cat, W, w.plan, nullptr, 0, med_outputs, nullptr, st);
            if (rc) return rc;
        }
        plan_queued = false;
        if (use_mean) {
            rc = launch_mean(&dirty, dev_spectrum, nb, n_cat, W, dev_median, dev_s_instr, dev_psd, grid->scale_log2, nullptr, nullptr, st);
        } else {
            rc = launch_median(dev_spectrum, nb, n_cat, W, dev_median, dev_s_instr, dev_psd, params->median_norm,
                               grid->scale_log2, &w.plan, nullptr, nullptr, nullptr, nullptr, st);
        }
        if (rc) return rc;
    }
    if (plan_queued) GBFG_CUDA(cudaStreamWaitEvent(st, side->ev_plan, 0));     // nothing of this call runs after it returns
    GBFG_CUDA(cudaMemcpyAsync(host, w.counters, sizeof(int64_t) * n_read_all, cudaMemcpyDeviceToHost, st));
    GBFG_CUDA(cudaStreamSynchronize(st));
    for (int c = 0; c < n_cat; ++c) {
        host_results[c].n_median_outputs = host[i_med + c];
        host_results[c].n_snr_tests = host[i_tests + c];
    }
    return GBFG_OK;
}

static int loop_impl(const gbfg_grid *grid, const double *dev_A, const double *dev_f,
                     const double *dev_fdot, const int64_t *offsets, int32_t n_cat,
                     const double *dev_s_instr, const gbfg_iter_params *params,
                     int64_t *dev_spectrum, int64_t *dev_median, double *dev_psd,
                     uint8_t *dev_resolved, gbfg_iter_result *host_results,
                     void *workspace, size_t workspace_bytes, void *stream, bool prepared,
                     cudaEvent_t records_ready = nullptr)
{
    int rc = loop_validate(grid, params);                  // argument errors are reported before any CUDA call
    if (rc) return rc;
    rc = bind_thread_to_current_device();
    if (rc) return rc;
    return drain_on_error(loop_body(grid, dev_A, dev_f, dev_fdot, offsets, n_cat, dev_s_instr, params, dev_spectrum, dev_median,
                                    dev_psd, dev_resolved, host_results, workspace, workspace_bytes, stream, prepared,
                                    records_ready), (cudaStream_t)stream);
}

extern "C" int gbfg_subtract_until_converged(const gbfg_grid *grid, const double *dev_A, const double *dev_f,
                                             const double *dev_fdot, const int64_t *offsets, int32_t n_cat,
                                             const double *dev_s_instr, const gbfg_iter_params *params,
                                             int64_t *dev_spectrum, int64_t *dev_median, double *dev_psd,
                                             uint8_t *dev_resolved, gbfg_iter_result *host_results,
                                             void *workspace, size_t workspace_bytes, void *stream)
{
    return loop_impl(grid, dev_A, dev_f, dev_fdot, offsets, n_cat, dev_s_instr, params, dev_spectrum, dev_median, dev_psd,
                     dev_resolved, host_results, workspace, workspace_bytes, stream, false);
}

// sample -> deposit -> loop.  The candidate records of the loop (a pass over the catalog against S_instr alone) are
// built on the side stream while the deposit runs: both only read the catalog.
static int simulate_body(const gbfg_grid *grid, const gbfg_pop *pops, const int64_t *offsets, int32_t n_cat,
                         uint64_t seed, const uint32_t *cat_ids, const double *dev_s_instr, const gbfg_iter_params *params,
                         double *dev_A, double *dev_f, double *dev_fdot,
                         int64_t *dev_total, int64_t *dev_spectrum, int64_t *dev_median, double *dev_psd,
                         uint8_t *dev_resolved, int64_t *dev_err_count, gbfg_iter_result *host_results,
                         void *workspace, size_t workspace_bytes, void *stream, EarlyOut *eo = nullptr)
{
    int rc = loop_validate(grid, params);
    if (rc) return rc;
    if (!offsets || n_cat < 1 || !dev_s_instr || !dev_spectrum || !dev_median || !dev_psd || !dev_resolved || !host_results)
        return GBFG_ERR_INVALID_ARG;
    CatTable ct;
    rc = make_cat_table(offsets, n_cat, &ct);
    if (rc) return rc;
    const int64_t n = ct.offsets[n_cat];
    if (!workspace || ((uintptr_t)workspace & 31u)) return GBFG_ERR_WORKSPACE;     // (256-bit accesses to its records)
    Workspace w = carve(workspace, grid->n_bins, n, n_cat);
    if (workspace_bytes < w.bytes) return GBFG_ERR_WORKSPACE;
    cudaStream_t st = (cudaStream_t)stream;
    SideStream *side = side_stream();
    if (!side) return set_cuda_error(cudaErrorMemoryAllocation, "side stream");
    const GridDev g = make_grid_dev(grid);
    const int64_t nb = grid->n_bins;
    const bool preselect = (params->flags & GBFG_FLAG_NO_PRESELECT) == 0;
    // side stream, next to the sampling: the prefix of 1/S_instr (after whatever the caller queued to produce S_instr)
    GBFG_CUDA(cudaEventRecord(side->ev_aux, st));
    GBFG_CUDA(cudaStreamWaitEvent(side->s, side->ev_aux, 0));
    rc = loop_prefix_s_instr(g, dev_s_instr, preselect, w, side->s);
    if (rc) return rc;
    GBFG_CUDA(cudaEventRecord(side->ev_noise, side->s));    // S_instr is on the device by now (gbfg_simulate_host copies it on this stream)
    const size_t row_bytes = sizeof(int64_t) * (size_t)n_cat * (size_t)nb;
    GBFG_CUDA(cudaMemsetAsync(dev_spectrum, 0, row_bytes, st));
    if (n > 0) GBFG_CUDA(cudaMemsetAsync(dev_resolved, 0, (size_t)n, st));
    rc = loop_init_workspace(w, nb, n_cat, st);
    if (rc) return rc;
    // stages (i) and (ii) in one kernel: every source is deposited by the thread that draws it (sample.cu).
    // Its stamps (-1) never equal those of the loop's subtractions (1 .. max_iter).
    // The catalog is drawn in a few pieces; the candidate records of a piece (a pass over its sources against S_instr
    // alone) are built on the side stream while the next piece is drawn: the drawing is bound by its arithmetic, the
    // pre-selection by L2 round trips, so the two share the SMs well.
    struct PieceCtx {
        const GridDev *g; const CatTable *ct; const double *A, *f, *fdot; const uint8_t *resolved; const double *s_instr;
        double rho_th; bool preselect; const Workspace *w; cudaStream_t st; SideStream *side;
    } pc = {&g, &ct, dev_A, dev_f, dev_fdot, dev_resolved, dev_s_instr, params->rho_th, preselect, &w, st, side};
    auto after_piece = [](void *ctx, int64_t i_begin, int64_t i_end) -> int {
        PieceCtx &p = *(PieceCtx *)ctx;
        GBFG_CUDA(cudaEventRecord(p.side->ev_aux, p.st));
        GBFG_CUDA(cudaStreamWaitEvent(p.side->s, p.side->ev_aux, 0));
        return cand_build_range(*p.g, *p.ct, p.A, p.f, p.fdot, p.resolved, p.preselect ? p.s_instr : nullptr, p.rho_th, nullptr,
                                p.w->sw, i_begin, i_end, p.side->s);
    };
    if (n > 0) {
        rc = cand_build_begin(ct, nb, w.sw, side->s);
        if (rc) return rc;
    }
    {
        SampleDeposit dep = {dev_spectrum, w.diff, dev_err_count, w.wide_flag, plain_marks(w, nb, -1), 0, nullptr, nullptr};
        dep.piece = n_cat == 1 ? (n + 3) / 4 : 0;               // a batch: catalog by catalog
        if (dep.piece < 1000000) dep.piece = dep.piece ? 1000000 : 0;
        dep.after_piece = after_piece;
        dep.ctx = &pc;
        rc = sample_catalog_ids(grid, pops, offsets, n_cat, 0u, cat_ids, seed, dev_A, dev_f, dev_fdot, stream, &dep);
        if (rc) return rc;
    }
    if (n > 0) {
        rc = cand_build_finish(g, ct, w.sw, side->s);
        if (rc) return rc;
    }
    GBFG_CUDA(cudaEventRecord(side->ev_aux, side->s));      // the records are ready
    // this stream: the scan of the wide sources' range updates into the spectrum
    rc = launch_scan(nb, n_cat, dev_spectrum, w.diff, w.tile_sums, w.wide_flag, plain_marks(w, nb, -1), st);
    if (rc) return rc;
    if (dev_total) GBFG_CUDA(cudaMemcpyAsync(dev_total, dev_spectrum, row_bytes, cudaMemcpyDeviceToDevice, st));
    GBFG_CUDA(cudaStreamWaitEvent(st, side->ev_noise, 0));  // the first estimator pass reads S_instr
    // the loop waits for the records (side->ev_aux) after its first estimator pass, which overlaps their build
    return loop_body(grid, dev_A, dev_f, dev_fdot, offsets, n_cat, dev_s_instr, params, dev_spectrum, dev_median, dev_psd,
                     dev_resolved, host_results, workspace, workspace_bytes, stream, true, side->ev_aux, eo);
}

extern "C" int gbfg_simulate(const gbfg_grid *grid, const gbfg_pop *pops, const int64_t *offsets, int32_t n_cat,
                             uint64_t seed, const uint32_t *cat_ids, const double *dev_s_instr, const gbfg_iter_params *params,
                             double *dev_A, double *dev_f, double *dev_fdot,
                             int64_t *dev_total, int64_t *dev_spectrum, int64_t *dev_median, double *dev_psd,
                             uint8_t *dev_resolved, int64_t *dev_err_count, gbfg_iter_result *host_results,
                             void *workspace, size_t workspace_bytes, void *stream)
{
    int rc = loop_validate(grid, params);
    if (rc) return rc;
    rc = bind_thread_to_current_device();
    if (rc) return rc;
    return drain_on_error(simulate_body(grid, pops, offsets, n_cat, seed, cat_ids, dev_s_instr, params, dev_A, dev_f, dev_fdot,
                                        dev_total, dev_spectrum, dev_median, dev_psd, dev_resolved, dev_err_count, host_results,
                                        workspace, workspace_bytes, stream), (cudaStream_t)stream);
}

// The path as the paper runs it (Fig. 3): Lambda of the paper's own population model -> catalog ->
// deposit -> loop (typically with the running mean of eq. D1 and the S_n stop rule) -> coarse-grained S_n and h_c.
extern "C" int gbfg_simulate_paper(const gbfg_grid *grid, const gbfg_pop_paper *pops, const int64_t *offsets, int32_t n_cat,
                                   uint64_t seed, const uint32_t *cat_ids, const double *dev_s_instr,
                                   const gbfg_iter_params *params, double *dev_A, double *dev_f, double *dev_fdot,
                                   int64_t *dev_total, int64_t *dev_spectrum, int64_t *dev_median, double *dev_psd,
                                   uint8_t *dev_resolved, int64_t *dev_err_count, gbfg_iter_result *host_results,
                                   const int64_t *dev_edges, int32_t n_coarse, double *dev_S_coarse, double *dev_f_coarse,
                                   double *dev_hc, void *workspace, size_t workspace_bytes, void *stream)
{
    int rc = loop_validate(grid, params);
    if (rc) return rc;
    if (!offsets || n_cat < 1 || !dev_s_instr || !dev_spectrum || !dev_median || !dev_psd || !dev_resolved || !host_results)
        return GBFG_ERR_INVALID_ARG;
    if ((dev_edges != nullptr) != (dev_S_coarse != nullptr) || (dev_edges && n_coarse < 1)) return GBFG_ERR_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    rc = sample_catalog_paper_ids(grid, pops, offsets, n_cat, 0u, cat_ids, seed, dev_A, dev_f, dev_fdot, stream);
    if (rc) return rc;
    const int64_t n = offsets[n_cat];
    const size_t row_bytes = sizeof(int64_t) * (size_t)n_cat * (size_t)grid->n_bins;
    GBFG_CUDA(cudaMemsetAsync(dev_spectrum, 0, row_bytes, st));
    if (n > 0) GBFG_CUDA(cudaMemsetAsync(dev_resolved, 0, (size_t)n, st));
    rc = gbfg_deposit(grid, dev_A, dev_f, dev_fdot, offsets, n_cat, nullptr, nullptr, +1, dev_spectrum, dev_err_count,
                      workspace, workspace_bytes, stream);
    if (rc) return rc;
    if (dev_total) GBFG_CUDA(cudaMemcpyAsync(dev_total, dev_spectrum, row_bytes, cudaMemcpyDeviceToDevice, st));
    rc = loop_impl(grid, dev_A, dev_f, dev_fdot, offsets, n_cat, dev_s_instr, params, dev_spectrum, dev_median, dev_psd,
                   dev_resolved, host_results, workspace, workspace_bytes, stream, false);
    if (rc) return rc;
    if (dev_edges) {                                        // eqs. (13)-(14), (B1): the datum the inference works with
        rc = gbfg_coarse_grain(dev_psd, grid->n_bins, n_cat, dev_edges, n_coarse, grid->f_min, grid->t_obs, dev_S_coarse,
                               dev_f_coarse, dev_hc, stream);
        if (rc) return rc;
        GBFG_CUDA(cudaStreamSynchronize(st));
    }
    return GBFG_OK;
}

extern "C" int gbfg_simulate_host(const gbfg_grid *grid, const gbfg_pop *pops, const int64_t *offsets, int32_t n_cat,
                                  uint64_t seed, const uint32_t *cat_ids, const double *host_s_instr, const gbfg_iter_params *params,
                                  double *host_psd, uint8_t *host_resolved, gbfg_iter_result *host_results)
{
    if (!valid_grid(grid) || !pops || !offsets || n_cat < 1 || !host_psd || !host_results)
        return GBFG_ERR_INVALID_ARG;
    if (n_cat > GBFG_MAX_CAT) return GBFG_ERR_UNSUPPORTED;
    int rc = check_device();
    if (rc) return rc;
    rc = bind_thread_to_current_device();
    if (rc) return rc;
    const int64_t n = offsets[n_cat];
    const size_t nb = (size_t)grid->n_bins, rows = (size_t)n_cat * nb;
    const size_t ws_bytes = gbfg_workspace_bytes(grid, n, n_cat);
    if (!ws_bytes) return GBFG_ERR_INVALID_ARG;
    // one allocation, carved
    size_t off = 0;
    auto take = [&](size_t bytes) { size_t o = off; off += (bytes + 255) & ~(size_t)255; return o; };
    const size_t nn = (size_t)(n > 0 ? n : 1);
    const size_t oA = take(8 * nn), oF = take(8 * nn), oD = take(8 * nn);
    const size_t oS = take(8 * rows), oM = take(8 * rows), oP = take(8 * rows), oI = take(8 * nb);
    const size_t oR = take(nn), oW = take(ws_bytes);
    // the device arena and the stream are kept between calls of the same host thread (gbfg_release_cached frees them)
    HostCallCache &cc = host_call_cache();
    int dev = 0;
    GBFG_CUDA(cudaGetDevice(&dev));
    if (cc.base && (cc.bytes < off || cc.device != dev)) { cudaFree(cc.base); cc.base = nullptr; cc.bytes = 0; }
    if (!cc.base) {
        GBFG_CUDA(cudaMalloc((void **)&cc.base, off));
        cc.bytes = off; cc.device = dev;
    }
    if (!cc.stream) {
        cudaError_t es = cudaStreamCreateWithFlags(&cc.stream, cudaStreamNonBlocking);
        if (es != cudaSuccess) { cc.stream = nullptr; return set_cuda_error(es, "cudaStreamCreate"); }
    }
    char *base = cc.base;
    cudaStream_t st = cc.stream;
    cudaError_t e;
    rc = GBFG_OK;
    // S_instr goes up on the loop's side stream, ahead of the candidate build gbfg_simulate queues there: the copy
    // runs while this stream samples and deposits, and gbfg_simulate joins the two streams before the loop reads it
    SideStream *side = side_stream();
    if (!side) return set_cuda_error(cudaErrorMemoryAllocation, "side stream");
    if (host_s_instr) {
        e = cudaMemcpyAsync(base + oI, host_s_instr, 8 * nb, cudaMemcpyHostToDevice, side->s);
        if (e != cudaSuccess) rc = set_cuda_error(e, "cudaMemcpyAsync(s_instr)");
    } else {
        // no curve given: the library's own (gbfg_instrument_noise), a function of the grid alone, made on the device
        rc = gbfg_instrument_noise(grid, (double *)(base + oI), side->s);
    }
    // the PSD may leave early (EarlyOut) when the caller's buffer is pinned host memory a kernel can store into
    EarlyOut eo = {host_psd, nullptr, 8 * rows, side->copy, -1, -1, 0, 0.0, host_resolved, (size_t)n, side->ev_copy, false};
    {
        cudaPointerAttributes at;
        if (cudaPointerGetAttributes(&at, host_psd) == cudaSuccess && at.type == cudaMemoryTypeHost && at.devicePointer)
            eo.host_psd_dev = (double *)at.devicePointer;
        (void)cudaGetLastError();
        // (a copy into pageable memory would hold the host up in the middle of the loop)
        if (!host_resolved || cudaPointerGetAttributes(&at, host_resolved) != cudaSuccess || at.type != cudaMemoryTypeHost)
            eo.host_resolved = nullptr;
        (void)cudaGetLastError();
    }
    if (!rc) {
        rc = loop_validate(grid, params);
        if (!rc)
            rc = drain_on_error(simulate_body(grid, pops, offsets, n_cat, seed, cat_ids, (const double *)(base + oI), params,
                                              (double *)(base + oA), (double *)(base + oF), (double *)(base + oD), nullptr,
                                              (int64_t *)(base + oS), (int64_t *)(base + oM), (double *)(base + oP),
                                              (uint8_t *)(base + oR), nullptr, host_results, base + oW, ws_bytes, st,
                                              eo.host_psd_dev ? &eo : nullptr), st);
    }
    if (!rc) {
        // nothing of the loop is in flight any more (it synchronises its stream before it returns)
        e = cudaSuccess;
        if (host_resolved && n > 0 && !eo.resolved_out)
            e = cudaMemcpyAsync(host_resolved, base + oR, (size_t)n, cudaMemcpyDeviceToHost, side->copy);
        if (e == cudaSuccess) {
            if (eo.started_after >= 0) {                        // the rest of the PSD, then what was stamped since the last patch
                if (eo.psd_sent < eo.bytes)
                    e = cudaMemcpyAsync((char *)host_psd + eo.psd_sent, base + oP + eo.psd_sent, eo.bytes - eo.psd_sent,
                                        cudaMemcpyDeviceToHost, side->copy);
                const Workspace w = carve(base + oW, grid->n_bins, n, n_cat);
                if (launch_psd_patch(eo, (const double *)(base + oP), w.blk_stamp, w.plan.n_dblk, w.plan.dblk_log2, grid->n_bins,
                                     n_cat, eo.patched_upto, 0x7fffffff) != GBFG_OK)
                    e = cudaErrorUnknown;
            } else {
                e = cudaMemcpyAsync(host_psd, base + oP, 8 * rows, cudaMemcpyDeviceToHost, st);
            }
        }
        if (e == cudaSuccess) e = cudaStreamSynchronize(st);
        if (e == cudaSuccess) e = cudaStreamSynchronize(side->copy);
        if (e != cudaSuccess) rc = set_cuda_error(e, "copy back");
    }
    cudaStreamSynchronize(side->copy);
    cudaStreamSynchronize(st);
    return rc;
}

extern "C" int gbfg_release_cached(void)
{
    release_thread_resources();
    return GBFG_OK;
}
