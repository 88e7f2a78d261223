// median.cu — stage (iii): exact running median of eq. (D2) + the PSD of eq. (10).
//
// DESIGN.md R3: odd window W = 2h+1 centred on k, ends reflected, statistic = the h-th smallest
// of the 2h+1 int64 values.  Only integer comparisons decide the result, so it is exact.
//
// Persistent CTAs (two of 512 threads per SM for the 32-bit-key kernel, median_kernel.cuh) take tiles of at
// most S = LT - 2h consecutive outputs — from the work list plan_kernel (below) derives from the blocks the
// last subtraction made dirty, or (stage call) from a static tiling of every row.  The tile and its two h-bin
// halos (Lt = outputs + 2h <= LT positions, rounded up to a multiple of the CTA width) are staged in shared
// memory and sorted ONCE by (value, position): an LSD radix sort, 8 bits per pass, that skips the passes whose
// digit is the same for the whole tile (spectrum values rarely need more than four).  The lanes of a warp that
// hold the same digit are found with eight warp reductions (a ballot each), not with match.any: the SM retires
// one MATCH every ~50 clocks, which made it the single slowest thing in the kernel.  With the sorted order in
// hand a window is a set of ranks, kept as a bitmap (one bit per rank), and its median is the (h+1)-th set bit:
//   * the bitmaps of 16 windows per tile (one per warp, evenly spaced) are built from the sorted positions: the
//     windows a position lies in are a range of warps (a 16-bit mask per lane), and a 32 x 32 bit transpose turns
//     the masks of two words of ranks into the bitmap words of all warps; the (h+1)-th set bit of each bitmap is
//     found by counting words;
//   * every warp then slides its window 32 outputs at a time.  Inside such a chunk lane i takes output j0 + i:
//     two popcounts of ballots (how many of the ranks that left / entered lie under the chunk's first median)
//     say how many window elements it must move, and in which direction; it moves word by word — 32 ranks and
//     typically 8 window elements per step, one popcount — testing positions only for the 64 "special" ranks
//     that enter or leave inside the chunk (a second bitmap marks them), and picks the bit in the last word.
//     Plateaus left by wide chirps (long stretches of out-of-window ranks) cost one step per 32 ranks.
// Every lane writes the median of its own output from inside that loop, fused with
//     psd[k] = s_instr[k] + C * (med[k] * 2^scale_log2)        (eqs. 10, D2, D3).
#include <mutex>

#include "median_kernel.cuh"

namespace gbfg {

__global__ void __launch_bounds__(256)
psd_kernel(const int64_t *__restrict__ med, const double *__restrict__ s_instr, int64_t n, double norm,
           double scale, double *__restrict__ psd)
{
    const int64_t row = (int64_t)blockIdx.y * n;
    int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    for (; k < n; k += stride) {
        double e = (double)med[row + k] * scale;
        psd[row + k] = s_instr[k] + norm * e;
    }
}

// ---------------------------------------------------------------------------------------------
// plan_kernel: one CTA per row.  Turns the dirty-block stamps of the last subtraction into
//   cum[row][b]  = number of dirty blocks before block b (b = 0 .. n_dblk), and
//   the work list of the running median: every maximal run of dirty blocks is cut into pieces of at
//   most S outputs (runs longer than one wave of CTAs are cut into a multiple of `wave` pieces).
// all_dirty != 0: every block counts as dirty (first iteration, cap branch without tracking).
// ctr[0] must be zero on entry; ctr[1] (the consumers' ticket) likewise.
// ---------------------------------------------------------------------------------------------
#ifdef PLAN_TIMING
#define PLAN_TICK(i) do { __syncthreads(); if (tid == 0 && blockIdx.x == 0) { const long long now_ = clock64(); if (i) a.dbg[i] += now_ - plan_t_prev; plan_t_prev = now_; } } while (0)
#else
#define PLAN_TICK(i) do { } while (0)
#endif
constexpr int PLAN_THREADS = 1024;
constexpr int PLAN_MIN_OUT = 512;              // outputs of the smallest tile the plan cuts

struct PlanArgs {
    const int *blk_stamp;   // [n_cat][n_dblk]
    int stamp;
    int all_dirty;
    int n_dblk, dblk_log2;
    int64_t n_bins;
    int S;                  // outputs per tile at most
    int wave;               // CTAs of one wave of the median kernel
    int *cum;               // [n_cat][n_dblk + 1]
    int *range;             // [n_cat][2]
    int4 *items;
    int *ctr;
    int max_items;
    int64_t *zero_ptr;      // per-iteration counters of the loop, cleared here (nullable)
    int zero_n;
    int64_t *out_count;     // [n_cat] outputs planned, accumulated (nullable)
    int *wide_ctr;          // [2] counter words of the wide list, cleared here
    unsigned long long *zero2_ptr;   // [n_cat] PSD-change words of the loop, cleared here (nullable)
    // the iteration's counters, handed to the host before they are cleared (nullable): pub_n words copied to
    // mapped pinned host memory, then the sequence number written behind them (the host polls it)
    const int64_t *pub_src;
    int64_t *pub_dst;
    int pub_n, pub_flag_at;
    int64_t pub_seq;
#ifdef PLAN_TIMING
    long long *dbg;         // probe builds only: clocks per phase, summed over launches, [16]
#endif
    int64_t *zero_sums;     // nullable: cleared here (PlanPublish)
    int zero_sums_n;
    int *near_fold;         // SnrWork::any_near (nullable): a near-threshold flag raised by the last test (word 1) becomes
                            // visible to the next one (word 0) here, between the two launches
};

// len < 2^31 (n_bins is): 32-bit divisions, the 64-bit ones are long instruction sequences
// shared memory: [n_dblk + 9] ints for the dirty words and their two prefixes (3 * ceil(n_dblk / 32) used), then the
// runs, 3 ints each, [n_dblk / 2 + 1]
static size_t plan_smem_bytes(int n_dblk) { return sizeof(int) * (size_t)((n_dblk + 9) + 3 * (n_dblk / 2 + 1)); }

__device__ __forceinline__ void plan_pieces(int64_t len64, int S, int wave, int *pieces, int *piece_len)
{
    const unsigned len = (unsigned)len64;
    unsigned np = (len + (unsigned)S - 1u) / (unsigned)S;
    if (np > (unsigned)wave) np = (np + (unsigned)wave - 1u) / (unsigned)wave * (unsigned)wave;
    const unsigned pl = (len + np - 1u) / np;
    *piece_len = (int)pl;
    *pieces = (int)((len + pl - 1u) / pl);
}

// The dirty flags of a row are kept as bits, 32 blocks per word (at most 512 words): cum comes from a scan of
// the words' popcounts, the runs from the words' rising and falling edges (the k-th start belongs to the k-th
// end), so that a late pass (a few hundred short runs) is a few thousand warp instructions on the one SM it runs on.
__global__ void __launch_bounds__(PLAN_THREADS)
plan_kernel(PlanArgs a)
{
    extern __shared__ int s_mem[];
    __shared__ int wtot[32];
    __shared__ int row_pieces, row_base, s_total;
    const unsigned FULL = 0xffffffffu;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int row = blockIdx.x;
    const int nb = a.n_dblk, nw = (nb + 31) >> 5;
    const int *st = a.blk_stamp ? a.blk_stamp + (int64_t)row * nb : nullptr;
    int *cum = a.cum + (int64_t)row * (nb + 1);
    unsigned *s_word = reinterpret_cast<unsigned *>(s_mem);   // [nw] dirty flags
    int *s_wpre = s_mem + nw;                                  // [nw] dirty blocks before the word
    int *s_rpre = s_mem + 2 * nw;                              // [nw] runs that start before the word
    int *s_run = s_mem + nb + 9;                               // (first block, end block, first piece) per run
#ifdef PLAN_TIMING
    long long plan_t_prev = 0;
#endif
    PLAN_TICK(0);
    if (tid == 0) row_pieces = 0;
    if (row == 0 && tid < 2) a.wide_ctr[tid] = 0;
    if (row == 0 && tid == 0 && a.near_fold && a.near_fold[1]) a.near_fold[0] = 1;
    // the stamps first: all of a thread's loads in flight while warp 0 hands the last pass's counters to the host
    constexpr int PLAN_LOADS = DIRTY_MAX_BLOCKS / PLAN_THREADS;
    static_assert(PLAN_LOADS * PLAN_THREADS == DIRTY_MAX_BLOCKS && PLAN_LOADS <= 16, "one round of loads covers a row");
    int v[PLAN_LOADS];
#pragma unroll
    for (int u = 0; u < PLAN_LOADS; ++u) {
        const int b = u * PLAN_THREADS + tid;
        v[u] = (!a.all_dirty && b < nb) ? st[b] : a.stamp;
    }
    if (row == 0 && warp == 0) {
        // What the pass before wrote (this kernel runs behind the SNR test) goes to the host by plain stores over
        // PCIe: no copy engine on the path.  One warp does it, and clears the counters behind its own loads, while
        // the others go on; the CTA meets again at the barrier below.
        if (a.pub_dst) for (int i = lane; i < a.pub_n; i += 32) a.pub_dst[i] = a.pub_src[i];
        __syncwarp();                                        // every lane has its values: the words may be cleared
        if (a.zero_ptr) for (int i = lane; i < a.zero_n; i += 32) a.zero_ptr[i] = 0;
        if (a.zero2_ptr) for (int i = lane; i < (int)gridDim.x; i += 32) a.zero2_ptr[i] = 0ull;
        if (a.pub_dst) {
            __threadfence_system();
            __syncwarp();
            if (lane == 0) *(volatile int64_t *)(a.pub_dst + a.pub_flag_at) = a.pub_seq;
        }
    }
    PLAN_TICK(1);
    if (row == 0 && a.zero_sums) for (int i = tid; i < a.zero_sums_n; i += PLAN_THREADS) a.zero_sums[i] = 0;
#pragma unroll
    for (int u = 0; u < PLAN_LOADS; ++u) {
        const int b = u * PLAN_THREADS + tid;
        const unsigned wd = __ballot_sync(FULL, b < nb && v[u] == a.stamp);
        if (lane == 0 && b < nb) s_word[b >> 5] = wd;
    }
    __syncthreads();
    PLAN_TICK(2);
    // per word: dirty blocks, run starts (a dirty block behind a clean one), run ends; one scan for both counts
    unsigned w = 0, starts = 0, ends = 0, open_in = 0;
    if (tid < nw) {
        w = s_word[tid];
        const unsigned prev = tid > 0 ? s_word[tid - 1] >> 31 : 0u;
        const unsigned next = tid + 1 < nw ? s_word[tid + 1] & 1u : 0u;
        starts = w & ~((w << 1) | prev);
        ends = w & ~((w >> 1) | (next << 31));
        open_in = prev & w & 1u;                              // a run crosses into this word
    }
    const int c = __popc(w);
    {
        const int packed = c | (__popc(starts) << 16);        // both totals stay under 2^16 (n_dblk <= 16384)
        int incl = packed;
        for (int o = 1; o < 32; o <<= 1) {
            const int up = __shfl_up_sync(FULL, incl, o);
            if (lane >= o) incl += up;
        }
        if (lane == 31) wtot[warp] = incl;
        __syncthreads();
        int excl = incl - packed;
        for (int k = 0; k < warp; ++k) excl += wtot[k];
        if (tid < nw) { s_wpre[tid] = excl & 0xffff; s_rpre[tid] = excl >> 16; }
        if (tid == PLAN_THREADS - 1) s_total = excl + packed;
    }
    __syncthreads();
    const int n_dirty = s_total & 0xffff, nr = s_total >> 16;
    PLAN_TICK(3);
#pragma unroll 4
    for (int b = tid; b <= nb; b += PLAN_THREADS) {
        const int wi = b >> 5;
        cum[b] = wi < nw ? s_wpre[wi] + __popc(s_word[wi] & ((1u << (b & 31)) - 1u)) : n_dirty;
    }
    PLAN_TICK(4);
    if (w) {                                                 // first / last dirty block of the row
        const int before = s_wpre[tid];
        if (before == 0) a.range[2 * row] = tid * 32 + __ffs(w) - 1;
        if (before + c == n_dirty) a.range[2 * row + 1] = tid * 32 + 31 - __clz(w);
    }
    if (tid == 0 && n_dirty == 0) { a.range[2 * row] = 1; a.range[2 * row + 1] = 0; }
    if (tid < nw) {
        int k = s_rpre[tid];
        for (unsigned m = starts; m; m &= m - 1u) s_run[3 * k++] = tid * 32 + __ffs(m) - 1;
        k = s_rpre[tid] - (int)open_in;                      // runs that ended before this word
        for (unsigned m = ends; m; m &= m - 1u) s_run[3 * k++ + 1] = tid * 32 + __ffs(m);
    }
    // Tile size of this row: S outputs at most, less when the dirty part of the row would not fill
    // the row's share of one wave of CTAs (the latency of a short tile is what the tail iterations pay).
    int S = a.S;
    {
        const unsigned dirty_out = (unsigned)n_dirty << a.dblk_log2;        // <= n_bins + one block
        int share = a.wave / (int)gridDim.x;
        if (share < 1) share = 1;
        unsigned s_fit = (dirty_out + (unsigned)share - 1u) / (unsigned)share;
        if (s_fit < (unsigned)PLAN_MIN_OUT) s_fit = PLAN_MIN_OUT;
        if (s_fit < (unsigned)S) S = (int)s_fit;
    }
    __syncthreads();
    PLAN_TICK(5);
    // the place of every run's pieces in the row's part of the list
    for (int r = tid; r < nr; r += PLAN_THREADS) {
        const int64_t first = (int64_t)s_run[3 * r] << a.dblk_log2;
        int64_t last = (int64_t)s_run[3 * r + 1] << a.dblk_log2;
        if (last > a.n_bins) last = a.n_bins;
        int pieces, piece_len;
        plan_pieces(last - first, S, a.wave, &pieces, &piece_len);
        s_run[3 * r + 2] = atomicAdd(&row_pieces, pieces);
    }
    __syncthreads();
    if (tid == 0) {
        if (a.out_count) {                               // dirty outputs of the row = dirty blocks, the last one clipped
            int64_t outs = (int64_t)n_dirty << a.dblk_log2;
            if (nb > 0 && ((s_word[nw - 1] >> ((nb - 1) & 31)) & 1u)) outs -= ((int64_t)nb << a.dblk_log2) - a.n_bins;
            a.out_count[row] += outs;
        }
        if (gridDim.x == 1) { row_base = 0; a.ctr[0] = row_pieces; a.ctr[1] = 0; }
        else row_base = atomicAdd(&a.ctr[0], row_pieces);
    }
    __syncthreads();
    PLAN_TICK(6);
    const int rb0 = row_base;
    for (int r = warp; r < nr; r += PLAN_THREADS / 32) {
        const int64_t first = (int64_t)s_run[3 * r] << a.dblk_log2;
        int64_t last = (int64_t)s_run[3 * r + 1] << a.dblk_log2;
        if (last > a.n_bins) last = a.n_bins;
        int pieces, piece_len;
        plan_pieces(last - first, S, a.wave, &pieces, &piece_len);
        const int base = rb0 + s_run[3 * r + 2];
        for (int i = lane; i < pieces; i += 32) {
            const int64_t o = first + (int64_t)i * piece_len;
            const int64_t n_out = (last - o < piece_len) ? last - o : piece_len;
            if (base + i < a.max_items) a.items[base + i] = make_int4(row, (int)o, (int)n_out, 0);
        }
    }
    PLAN_TICK(7);
}

#ifdef PLAN_TIMING
static long long *plan_timing_words()
{
    static long long *p = nullptr;
    if (!p) { cudaMalloc(&p, 16 * sizeof(long long)); cudaMemset(p, 0, 16 * sizeof(long long)); }
    return p;
}
extern "C" void gbfg_debug_plan_timing(long long *out)
{
    cudaDeviceSynchronize();
    cudaMemcpy(out, plan_timing_words(), 16 * sizeof(long long), cudaMemcpyDeviceToHost);
    cudaMemset(plan_timing_words(), 0, 16 * sizeof(long long));
}
#endif

int median_tile_outputs(int window) { return MED_LT32 - (window - 1); }

int median_tiles(int64_t n_bins, int window)
{
    int S = MED_LT32 - (window - 1);
    return (int)((n_bins + S - 1) / S);
}

// upper bound of the number of work items plan_kernel can emit for one row
int median_max_items(int64_t n_bins)
{
    const int s_min = MED_LT32 - (GBFG_MAX_WINDOW - 1);
    const int s_small = s_min < PLAN_MIN_OUT ? s_min : PLAN_MIN_OUT;
    return dirty_blocks_per_row(n_bins) + 2 * (int)((n_bins + s_small - 1) / s_small) + 16;
}

// work list + cum from the stamps (blk_stamp NULL or all_dirty: everything)
int launch_plan(const int *blk_stamp, int stamp, bool all_dirty, int64_t n_bins, int n_cat, int window,
                const MedianPlan &pl, int64_t *zero_ptr, int zero_n, int64_t *out_count, unsigned long long *zero2_ptr,
                cudaStream_t st, const PlanPublish *pub)
{
    PlanArgs a;
    if (pub) { a.pub_src = pub->src; a.pub_dst = pub->dst; a.pub_n = pub->n; a.pub_flag_at = pub->flag_at; a.pub_seq = pub->seq; }
    else { a.pub_src = nullptr; a.pub_dst = nullptr; a.pub_n = 0; a.pub_flag_at = 0; a.pub_seq = 0; }
    a.zero_sums = pub ? pub->zero_sums : nullptr; a.zero_sums_n = pub ? pub->zero_sums_n : 0;
#ifdef PLAN_TIMING
    a.dbg = plan_timing_words();
#endif
    a.zero2_ptr = zero2_ptr;
    a.near_fold = pl.near_fold;
    a.zero_ptr = zero_ptr; a.zero_n = zero_n; a.out_count = out_count;
    a.blk_stamp = blk_stamp; a.stamp = stamp; a.all_dirty = (all_dirty || !blk_stamp) ? 1 : 0;
    a.n_dblk = pl.n_dblk; a.dblk_log2 = pl.dblk_log2; a.n_bins = n_bins;
    a.S = MED_LT32 - (window - 1);
    a.wave = 2 * sm_count();                             // two CTAs of the 32-bit-key kernel per SM
    a.wide_ctr = pl.wide_ctr;
    a.cum = pl.cum; a.range = pl.range; a.items = pl.items; a.ctr = pl.ctr; a.max_items = pl.max_items;
    const size_t smem = plan_smem_bytes(pl.n_dblk);
    static thread_local int attr_dev = -1;
    int dev = 0;
    GBFG_CUDA(cudaGetDevice(&dev));
    if (attr_dev != dev) {
        GBFG_CUDA(cudaFuncSetAttribute(plan_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                       (int)plan_smem_bytes(DIRTY_MAX_BLOCKS)));
        attr_dev = dev;
    }
    if (n_cat > 1) GBFG_CUDA(cudaMemsetAsync(pl.ctr, 0, 2 * sizeof(int), st));   // one row: the kernel sets both words
    {
        LaunchTimer lt(K_AUX, st);
        plan_kernel<<<n_cat, PLAN_THREADS, smem, st>>>(a);
    }
    GBFG_LAUNCH_CHECK("plan_kernel");
    return GBFG_OK;
}

// internal entry: median (+ PSD when psd != NULL).  plan != NULL: the tiles of its work list (made by
// launch_plan on the same stream); NULL: every row, statically tiled, and wide_items / wide_ctr give the
// room for the wide list ([tiles of the call] int4, 2 ints zeroed here).  neg_flag nullable: raised when
// a median is negative.  Two launches: the 32-bit-key kernel, two CTAs per SM, then the 64-bit-key kernel
// on the tiles the first one could not order (none for spectra in units of 2^-140 strain^2).
int median_static_tiles(int64_t n_bins, int n_cat, int window, int *S_out)
{
    const int s_max = MED_LT32 - (window - 1);
    const int slots = 2 * sm_count();
    int64_t tiles = (n_bins + s_max - 1) / s_max;
    if (tiles * n_cat > slots && n_cat == 1) tiles = (tiles + slots - 1) / slots * slots;   // whole waves of CTAs
    const int S = (int)((n_bins + tiles - 1) / tiles);
    if (S_out) *S_out = S;
    return (int)((n_bins + S - 1) / S);
}

#ifdef MED_TIMING
// probe builds (-DMED_TIMING): clocks per phase of the tile loop, [CTA][16], summed over the CTA's tiles and over the
// launches since the last read
static long long *median_timing_words()
{
    static long long *p = nullptr;
    if (!p) { cudaMalloc(&p, 1024 * 16 * sizeof(long long)); cudaMemset(p, 0, 1024 * 16 * sizeof(long long)); }
    return p;
}
extern "C" void gbfg_debug_median_timing(long long *out, int n_cta)
{
    cudaDeviceSynchronize();
    cudaMemcpy(out, median_timing_words(), (size_t)n_cta * 16 * sizeof(long long), cudaMemcpyDeviceToHost);
    cudaMemset(median_timing_words(), 0, 1024 * 16 * sizeof(long long));
}
#endif

int launch_median(const int64_t *x, int64_t n_bins, int n_cat, int window, int64_t *med,
                  const double *s_instr, double *psd, double norm, int scale_log2,
                  const MedianPlan *plan, int4 *wide_items, int *wide_ctr, int *neg_flag,
                  unsigned long long *delta_bits, cudaStream_t st)
{
    MedianArgs a;
#ifdef MED_TIMING
    a.dbg = median_timing_words();
#endif
    a.delta_bits = delta_bits;
    a.x = x; a.med = med; a.s_instr = s_instr; a.psd = psd; a.neg_flag = neg_flag;
    a.items = plan ? plan->items : nullptr; a.ctr = plan ? plan->ctr : nullptr; a.n_cat = n_cat;
    a.wide_items = plan ? plan->wide_items : wide_items;
    a.wide_ctr = plan ? plan->wide_ctr : wide_ctr;
    a.n = n_bins; a.h = window / 2;
    a.tiles = median_static_tiles(n_bins, n_cat, window, &a.S);
    a.norm = norm; a.scale = ldexp(1.0, scale_log2);
    constexpr size_t smem32 = median_smem_bytes<uint32_t, 512, MED_LT32>(), smem64 = median_smem_bytes<uint64_t, 1024, MED_LT64>();
    static thread_local int attr_dev = -1;
    int dev = 0;
    GBFG_CUDA(cudaGetDevice(&dev));
    if (attr_dev != dev) {
        GBFG_CUDA(cudaFuncSetAttribute(running_median_tile_kernel<uint32_t, 512, MED_LT32, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem32));
        GBFG_CUDA(cudaFuncSetAttribute(running_median_tile_kernel<uint64_t, 1024, MED_LT64, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem64));
        GBFG_CUDA(cudaFuncSetAttribute(running_median_tile_kernel<uint32_t, 512, MED_LT32, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem32));
        GBFG_CUDA(cudaFuncSetAttribute(running_median_tile_kernel<uint64_t, 1024, MED_LT64, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem64));
        attr_dev = dev;
    }
    const int sms = sm_count();
    if (!plan) GBFG_CUDA(cudaMemsetAsync(a.wide_ctr, 0, 2 * sizeof(int), st));     // plan_kernel clears them otherwise
    int64_t grid = plan ? 2 * sms : (int64_t)a.tiles * n_cat;
    if (grid > 2 * sms) grid = 2 * sms;
    LaunchTimer lt(K_MEDIAN, st);
    if (delta_bits) running_median_tile_kernel<uint32_t, 512, MED_LT32, true><<<(int)grid, 512, smem32, st>>>(a);
    else running_median_tile_kernel<uint32_t, 512, MED_LT32, false><<<(int)grid, 512, smem32, st>>>(a);
    GBFG_LAUNCH_CHECK("running_median_tile_kernel<u32>");
    a.items = a.wide_items; a.ctr = a.wide_ctr;
    a.wide_items = nullptr; a.wide_ctr = nullptr;
    if (grid > sms) grid = sms;
    cudaError_t e = delta_bits
        ? launch_dependent(running_median_tile_kernel<uint64_t, 1024, MED_LT64, true>, dim3((unsigned)grid), dim3(1024), smem64, st, a)
        : launch_dependent(running_median_tile_kernel<uint64_t, 1024, MED_LT64, false>, dim3((unsigned)grid), dim3(1024), smem64, st, a);
    if (e != cudaSuccess) return set_cuda_error(e, "running_median_tile_kernel<u64>");
    GBFG_LAUNCH_CHECK("running_median_tile_kernel<u64>");
    return GBFG_OK;
}

}  // namespace gbfg

using namespace gbfg;

// room for the list of tiles the 32-bit-key kernel leaves to the 64-bit-key one: 16 bytes of counters + one int4 per tile
extern "C" size_t gbfg_running_median_workspace_bytes(int64_t n_bins, int32_t n_cat, int32_t window)
{
    if (window < 1 || (window & 1) == 0 || window > GBFG_MAX_WINDOW || n_cat < 1 || n_cat > GBFG_MAX_CAT || n_bins < 1 ||
        n_bins >= 2147483648ll)
        return 0;
    const int s_max = MED_LT32 - (window - 1);
    const size_t tiles = (size_t)((n_bins + s_max - 1) / s_max) + 2 * 148 * 4;     // whole waves of CTAs on any part
    return 256 + sizeof(int4) * tiles * (size_t)n_cat;
}

extern "C" int gbfg_running_median(const int64_t *dev_spectrum, int64_t n_bins, int32_t n_cat, int32_t window,
                                   int64_t *dev_median_out, void *workspace, size_t workspace_bytes, void *stream)
{
    if (!dev_spectrum || !dev_median_out || dev_spectrum == dev_median_out) return GBFG_ERR_INVALID_ARG;
    if (window < 1 || (window & 1) == 0 || n_cat < 1 || n_bins < 1 || n_bins >= 2147483648ll) return GBFG_ERR_INVALID_ARG;
    if (window > GBFG_MAX_WINDOW || n_cat > GBFG_MAX_CAT) return GBFG_ERR_UNSUPPORTED;
    if (n_bins < window / 2 + 1) return GBFG_ERR_INVALID_ARG;
    if (!workspace || ((uintptr_t)workspace & 15)) return GBFG_ERR_WORKSPACE;
    const int tiles = median_static_tiles(n_bins, n_cat, window, nullptr);
    if (workspace_bytes < 256 + sizeof(int4) * (size_t)tiles * (size_t)n_cat) return GBFG_ERR_WORKSPACE;
    int rc = check_device();
    if (rc) return rc;
    // the caller's workspace holds the wide list (tiles whose values differ in their high 32 bits)
    char *tmp = (char *)workspace;
    return launch_median(dev_spectrum, n_bins, n_cat, window, dev_median_out, nullptr, nullptr, 1.0, 0, nullptr,
                         (int4 *)(tmp + 256), (int *)tmp, nullptr, nullptr, (cudaStream_t)stream);
}

// ---- gbfg_running_median_static: the same two kernels with the wide list in a file-scope device array, for callers that
// cannot allocate and have no workspace.  In host code the array's name is a host-side stand-in, not a device address
// (a kernel handed it would fault, or use the wrong memory): the address comes from cudaGetSymbolAddress, once per
// device, with that device current.  Every call shares the array; calls that overlap on the GPU race (include/gbfg.h).
static __device__ __align__(256) unsigned char g_median_static_scratch[GBFG_STATIC_SCRATCH_BYTES];

static int median_static_setup(void **scratch)
{
    static std::mutex mu;
    static void *ptr_of[64];                             // the array's address on each device
    int dev = 0;
    GBFG_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= 64) return GBFG_ERR_ARCH;
    std::lock_guard<std::mutex> lock(mu);
    if (!ptr_of[dev]) {
        void *ptr = nullptr;
        GBFG_CUDA(cudaGetSymbolAddress(&ptr, g_median_static_scratch));
        GBFG_CUDA(cudaFuncSetAttribute(running_median_tile_kernel<uint32_t, 512, MED_LT32, false>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                       (int)median_smem_bytes<uint32_t, 512, MED_LT32>()));
        GBFG_CUDA(cudaFuncSetAttribute(running_median_tile_kernel<uint64_t, 1024, MED_LT64, false>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                       (int)median_smem_bytes<uint64_t, 1024, MED_LT64>()));
        ptr_of[dev] = ptr;
    }
    *scratch = ptr_of[dev];
    return GBFG_OK;
}

extern "C" int gbfg_running_median_static(const int64_t *dev_spectrum, int64_t n_bins, int32_t n_cat, int32_t window,
                                          int64_t *dev_median_out, void *stream)
{
    if (!dev_spectrum || !dev_median_out || dev_spectrum == dev_median_out) return GBFG_ERR_INVALID_ARG;
    if (window < 1 || (window & 1) == 0 || n_cat < 1 || n_bins < 1 || n_bins >= 2147483648ll) return GBFG_ERR_INVALID_ARG;
    if (window > GBFG_MAX_WINDOW || n_cat > GBFG_MAX_CAT) return GBFG_ERR_UNSUPPORTED;
    if (n_bins < window / 2 + 1) return GBFG_ERR_INVALID_ARG;
    int rc = check_device();
    if (rc) return rc;
    MedianArgs a;
#ifdef MED_TIMING
    a.dbg = median_timing_words();
#endif
    a.tiles = median_static_tiles(n_bins, n_cat, window, &a.S);
    if ((int64_t)a.tiles * n_cat > (int64_t)GBFG_STATIC_MAX_TILES) return GBFG_ERR_STATIC_LIMIT;     // nothing launched
    void *scratch = nullptr;
    rc = median_static_setup(&scratch);
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    a.x = dev_spectrum; a.med = dev_median_out; a.s_instr = nullptr; a.psd = nullptr; a.neg_flag = nullptr; a.delta_bits = nullptr;
    a.items = nullptr; a.ctr = nullptr; a.n_cat = n_cat;
    a.wide_ctr = (int *)scratch;                         // [0] tiles in the list, [1] the consumers' ticket
    a.wide_items = (int4 *)((char *)scratch + 256);
    a.n = n_bins; a.h = window / 2;
    a.norm = 1.0; a.scale = 1.0;
    // the array keeps the last call's contents: the two counters start at zero, the list is written before it is read
    GBFG_CUDA(cudaMemsetAsync(a.wide_ctr, 0, 2 * sizeof(int), st));
    const int sms = sm_count();
    int64_t grid = (int64_t)a.tiles * n_cat;
    if (grid > 2 * sms) grid = 2 * sms;
    running_median_tile_kernel<uint32_t, 512, MED_LT32, false><<<(int)grid, 512, median_smem_bytes<uint32_t, 512, MED_LT32>(), st>>>(a);
    GBFG_LAUNCH_CHECK("running_median_tile_kernel<u32> (static scratch)");
    a.items = a.wide_items; a.ctr = a.wide_ctr;
    a.wide_items = nullptr; a.wide_ctr = nullptr;
    if (grid > sms) grid = sms;
    cudaError_t e = launch_dependent(running_median_tile_kernel<uint64_t, 1024, MED_LT64, false>, dim3((unsigned)grid), dim3(1024),
                                     median_smem_bytes<uint64_t, 1024, MED_LT64>(), st, a);
    if (e != cudaSuccess) return set_cuda_error(e, "running_median_tile_kernel<u64> (static scratch)");
    GBFG_LAUNCH_CHECK("running_median_tile_kernel<u64> (static scratch)");
    return GBFG_OK;
}

extern "C" int gbfg_psd(const int64_t *dev_median, const double *dev_s_instr, int64_t n_bins, int32_t n_cat,
                        double median_norm, int32_t scale_log2, double *dev_psd, void *stream)
{
    if (!dev_median || !dev_s_instr || !dev_psd) return GBFG_ERR_INVALID_ARG;
    if (n_cat < 1 || n_bins < 1 || scale_log2 < -1000 || scale_log2 > 0) return GBFG_ERR_INVALID_ARG;
    if (n_cat > GBFG_MAX_CAT) return GBFG_ERR_UNSUPPORTED;
    int rc = check_device();
    if (rc) return rc;
    int bx = (int)((n_bins + 255) / 256);
    int cap = sm_count() * 8;
    if (bx > cap) bx = cap;
    {
        LaunchTimer lt(K_PSD, (cudaStream_t)stream);
        psd_kernel<<<dim3(bx, n_cat), 256, 0, (cudaStream_t)stream>>>(dev_median, dev_s_instr, n_bins, median_norm,
                                                                       ldexp(1.0, scale_log2), dev_psd);
    }
    GBFG_LAUNCH_CHECK("psd_kernel");
    return GBFG_OK;
}

