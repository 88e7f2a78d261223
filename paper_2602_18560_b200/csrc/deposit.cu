// deposit.cu — stages (ii) and (v): spectrum[k] += sign * q_i over the bins a source's chirp covers.
//
// DESIGN.md R2 fixes the arithmetic.  The accumulator is int64, so any order and any regrouping of
// the additions gives the same bits.  That is used twice:
//   * narrow sources (w_eff <= NARROW) add q straight into the spectrum with 64-bit L2 atomics;
//   * wide sources use the range-update form: +q at k0 and -q at k0+w_eff in a difference array,
//     followed by one inclusive scan that is added into the spectrum (2 updates per source instead
//     of w; chirps reach 7e4 bins at 4 yr).  sum_k spectrum[k] is identical bit for bit.
// The scan is a two-launch tile scan (sums of the tiles that hold updates -> every tile adds up the
// sums before it, rescans and adds); the difference array is zeroed again on the way so the
// workspace is reusable.  Scan tiles that hold no update and start from a zero running value are
// skipped (stamps written by the deposit kernel).
// A subtraction also stamps the dirty blocks (gbfg_common.cuh) whose running-median outputs see a
// changed bin, so that stages (iii) and (iv) redo only those (DepositMarks).
#include "gbfg_common.cuh"

namespace gbfg {

constexpr int NARROW = DEP_NARROW;   // <= NARROW bins: direct atomics
constexpr int SCAN_THREADS = 256;
constexpr int SCAN_ITEMS = 8;        // int64 per thread
constexpr int SCAN_TILE = SCAN_THREADS * SCAN_ITEMS;
static_assert(SCAN_TILE == DEP_SCAN_TILE, "snr.cu stamps scan tiles of this size");

// One thread per addressed source.  `wide_flag` is set if any source used the difference array.
__global__ void __launch_bounds__(256)
deposit_kernel(GridDev g, CatTable ct, const double *__restrict__ A, const double *__restrict__ f,
               const double *__restrict__ fdot, const int64_t *__restrict__ sel_idx,
               const int64_t *__restrict__ sel_count, int64_t n_all, int32_t sign,
               int64_t *__restrict__ spectrum, int64_t *__restrict__ diff,
               int64_t *__restrict__ err_count, int *__restrict__ wide_flag, DepositMarks mk)
{
    const int64_t n = sel_idx ? *sel_count : n_all;
    int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    int rejected = 0;
    for (; t < n; t += stride) {
        const int64_t i = sel_idx ? sel_idx[t] : t;
        SrcBins s = source_bins(g, A[i], f[i], fdot[i]);
        if (s.status) { ++rejected; continue; }
        const int cat = cat_of(ct, i);
        const int64_t row = (int64_t)cat * g.n_bins;
        const int64_t v = sign >= 0 ? s.q : -s.q;
        if (v == 0) continue;
        deposit_one(s, v, g.n_bins, cat, spectrum + row, diff + row, wide_flag, mk);
    }
    if (err_count) {
        // warp-aggregate the reject count
        for (int o = 16; o; o >>= 1) rejected += __shfl_down_sync(0xffffffffu, rejected, o);
        if ((threadIdx.x & 31) == 0 && rejected) atomic_add_i64(err_count, rejected);
    }
}

// 256-bit global accesses (sm_100): one 32-byte sector per thread and instruction; p must be 32-byte aligned
__device__ __forceinline__ void ld_global_256(const int64_t *p, int64_t *v)
{
    asm volatile("ld.global.v4.s64 {%0, %1, %2, %3}, [%4];" : "=l"(v[0]), "=l"(v[1]), "=l"(v[2]), "=l"(v[3]) : "l"(p) : "memory");
}
__device__ __forceinline__ void st_global_256(int64_t *p, const int64_t *v)
{
    asm volatile("st.global.v4.s64 [%0], {%1, %2, %3, %4};" ::"l"(p), "l"(v[0]), "l"(v[1]), "l"(v[2]), "l"(v[3]) : "memory");
}

// phase 1: sums of the tiles of the difference array that hold an update (the others are not touched:
// their sum is zero by definition, whatever tile_sums holds from an earlier call).
// grid = (tiles_per_row, n_cat)
__global__ void __launch_bounds__(SCAN_THREADS)
scan_tile_sums_kernel(const int64_t *__restrict__ diff, int64_t n_bins, int tiles_per_row,
                      int64_t *__restrict__ tile_sums, const int *__restrict__ wide_flag,
                      const int *__restrict__ scan_stamp, int stamp)
{
    gbfg_let_next_kernel_start();
    if (*wide_flag != stamp) return;
    const int64_t ti = (int64_t)blockIdx.y * tiles_per_row + blockIdx.x;
    if (scan_stamp[ti] != stamp) return;
    __shared__ int64_t warp_sum[SCAN_THREADS / 32];
    const int64_t row = (int64_t)blockIdx.y * n_bins;
    const int64_t base = (int64_t)blockIdx.x * SCAN_TILE;
    int64_t acc = 0;
#pragma unroll
    for (int j = 0; j < SCAN_ITEMS; ++j) {
        int64_t k = base + (int64_t)j * SCAN_THREADS + threadIdx.x;
        if (k < n_bins) acc += diff[row + k];
    }
    for (int o = 16; o; o >>= 1) acc += __shfl_down_sync(0xffffffffu, acc, o);
    if ((threadIdx.x & 31) == 0) warp_sum[threadIdx.x >> 5] = acc;
    __syncthreads();
    if (threadIdx.x == 0) {
        int64_t t = 0;
        for (int w = 0; w < SCAN_THREADS / 32; ++w) t += warp_sum[w];
        tile_sums[ti] = t;
    }
}

// phase 2: every CTA adds up the sums of the stamped tiles before its own (a few thousand L2 reads:
// cheaper than a separate scan launch or a ticket per tile), rescans its tile, adds the running value
// into the spectrum and zeroes the difference array.
__global__ void __launch_bounds__(SCAN_THREADS)
scan_add_kernel(int64_t *__restrict__ diff, int64_t n_bins, int tiles_per_row,
                const int64_t *__restrict__ tile_sums, int64_t *__restrict__ spectrum,
                const int *__restrict__ wide_flag, const int *__restrict__ scan_stamp, int stamp)
{
    gbfg_wait_prior_kernel();                           // the tile sums
    if (*wide_flag != stamp) return;
    __shared__ int64_t warp_tot[SCAN_THREADS / 32];
    __shared__ int64_t tile_offset;
    const int64_t t0 = (int64_t)blockIdx.y * tiles_per_row;
    {
        // (every look-up of a thread in flight at once: a CTA far into the row would otherwise wait for two dependent
        // L2 round trips per 256 tiles before it)
        int64_t acc = 0;
        for (int tb = 0; tb < (int)blockIdx.x; tb += 8 * SCAN_THREADS) {
            int stp[8];
            int64_t sum[8];
#pragma unroll
            for (int u = 0; u < 8; ++u) {
                const int t = tb + u * SCAN_THREADS + threadIdx.x;
                stp[u] = t < (int)blockIdx.x ? scan_stamp[t0 + t] : stamp - 1;
            }
#pragma unroll
            for (int u = 0; u < 8; ++u) {
                const int t = tb + u * SCAN_THREADS + threadIdx.x;
                sum[u] = stp[u] == stamp ? tile_sums[t0 + t] : 0;
            }
#pragma unroll
            for (int u = 0; u < 8; ++u) acc += sum[u];
        }
        for (int o = 16; o; o >>= 1) acc += __shfl_down_sync(0xffffffffu, acc, o);
        if ((threadIdx.x & 31) == 0) warp_tot[threadIdx.x >> 5] = acc;
        __syncthreads();
        if (threadIdx.x == 0) {
            int64_t s = 0;
            for (int w = 0; w < SCAN_THREADS / 32; ++w) s += warp_tot[w];
            tile_offset = s;
        }
        __syncthreads();
    }
    // nothing to add in a tile without updates that starts from a zero running value
    if (scan_stamp[t0 + blockIdx.x] != stamp && tile_offset == 0) return;
    const int64_t row = (int64_t)blockIdx.y * n_bins;
    const int64_t base = (int64_t)blockIdx.x * SCAN_TILE + (int64_t)threadIdx.x * SCAN_ITEMS;
    // A thread's SCAN_ITEMS = 8 consecutive bins are two 32-byte sectors: moved as 256-bit vectors where the row
    // starts on a 32-byte boundary, a sector is touched once (with 64-bit accesses every load instruction of the warp
    // touches 32 sectors and every sector is touched four times: the kernel was bound by that).
    static_assert(SCAN_ITEMS == 8, "two 256-bit vectors per thread");
    const bool vec = ((((uintptr_t)(diff + row)) | ((uintptr_t)(spectrum + row))) & 31u) == 0 && base + SCAN_ITEMS <= n_bins;
    int64_t v[SCAN_ITEMS];
    int64_t tsum = 0;
    if (vec) {
        ld_global_256(diff + row + base, v);
        ld_global_256(diff + row + base + 4, v + 4);
#pragma unroll
        for (int j = 0; j < SCAN_ITEMS; ++j) tsum += v[j];
    } else {
#pragma unroll
        for (int j = 0; j < SCAN_ITEMS; ++j) {
            int64_t k = base + j;
            v[j] = k < n_bins ? diff[row + k] : 0;
            tsum += v[j];
        }
    }
    int64_t incl = tsum;
    for (int o = 1; o < 32; o <<= 1) {
        int64_t up = __shfl_up_sync(0xffffffffu, incl, o);
        if ((threadIdx.x & 31) >= o) incl += up;
    }
    __syncthreads();
    if ((threadIdx.x & 31) == 31) warp_tot[threadIdx.x >> 5] = incl;
    __syncthreads();
    int64_t run = tile_offset + incl - tsum;
    for (int w = 0; w < (threadIdx.x >> 5); ++w) run += warp_tot[w];
    if (vec) {
#pragma unroll
        for (int half = 0; half < 2; ++half) {
            int64_t r[4];
            int64_t any_r = 0, any_v = 0;
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                run += v[4 * half + j];
                r[j] = run;
                any_r |= run;
                any_v |= v[4 * half + j];
            }
            int64_t *const sp = spectrum + row + base + 4 * half;
            if (any_r != 0) {                               // (a bin whose running value is zero gets its own value back)
                int64_t s4[4];
                ld_global_256(sp, s4);
#pragma unroll
                for (int j = 0; j < 4; ++j) s4[j] += r[j];
                st_global_256(sp, s4);
            }
            if (any_v != 0) {
                const int64_t z[4] = {0, 0, 0, 0};
                st_global_256(diff + row + base + 4 * half, z);
            }
        }
        return;
    }
#pragma unroll
    for (int j = 0; j < SCAN_ITEMS; ++j) {
        int64_t k = base + j;
        run += v[j];
        if (k < n_bins) {
            if (run != 0) spectrum[row + k] += run;
            if (v[j] != 0) diff[row + k] = 0;
        }
    }
}

// ---------------------------------------------------------------------------------------------
// internal entry used by the stage call and by the loop.  diff: [n_cat*n_bins] zero on entry and
// on exit; tile_sums: [n_cat*tiles_per_row]; wide_flag: one int that must differ from mk.stamp on
// entry (it is left equal to it when a wide source was seen).
// mk.scan_stamp: [n_cat*tiles_per_row] ints, none equal to mk.stamp on entry.
// ---------------------------------------------------------------------------------------------
int scan_tiles_per_row(int64_t n_bins) { return (int)((n_bins + SCAN_TILE - 1) / SCAN_TILE); }

int launch_scan(int64_t n_bins, int n_cat, int64_t *spectrum, int64_t *diff, int64_t *tile_sums, int *wide_flag,
                const DepositMarks &mk, cudaStream_t st);

int launch_deposit(const GridDev &g, const CatTable &ct, const double *A, const double *f, const double *fdot,
                   const int64_t *sel_idx, const int64_t *sel_count, int64_t n_launch, int32_t sign,
                   int64_t *spectrum, int64_t *err_count, int64_t *diff, int64_t *tile_sums, int *wide_flag,
                   const DepositMarks &mk, cudaStream_t st, cudaEvent_t after_deposit)
{
    if (n_launch <= 0) {
        if (after_deposit) GBFG_CUDA(cudaEventRecord(after_deposit, st));
        return GBFG_OK;
    }
    int64_t blocks = (n_launch + 255) / 256;
    int64_t cap = (int64_t)sm_count() * 16;
    if (blocks > cap) blocks = cap;
    {
        LaunchTimer lt(K_DEPOSIT, st);
        deposit_kernel<<<(int)blocks, 256, 0, st>>>(g, ct, A, f, fdot, sel_idx, sel_count, ct.offsets[ct.n_cat], sign,
                                                    spectrum, diff, err_count, wide_flag, mk);
    }
    GBFG_LAUNCH_CHECK("deposit_kernel");
    if (after_deposit) GBFG_CUDA(cudaEventRecord(after_deposit, st));   // the stamps are written: the plan may start
    return launch_scan(g.n_bins, ct.n_cat, spectrum, diff, tile_sums, wide_flag, mk, st);
}

// the scan of the difference array into the spectrum (no-op unless wide_flag holds mk.stamp)
int launch_scan(int64_t n_bins, int n_cat, int64_t *spectrum, int64_t *diff, int64_t *tile_sums, int *wide_flag,
                const DepositMarks &mk, cudaStream_t st)
{
    const int tiles = scan_tiles_per_row(n_bins);
    dim3 grid(tiles, n_cat);
    LaunchTimer lt_scan(K_SCAN, st);     // the two scan kernels, as one
    if (mk.live_sums) {
        // whoever wrote the range updates kept the tile sums as well (the loop's test): the second kernel alone, and not as
        // a programmatic dependent of that test (its 1843 CTAs would sit on the SMs waiting while the test still runs)
        scan_add_kernel<<<grid, SCAN_THREADS, 0, st>>>(diff, n_bins, tiles, (const int64_t *)mk.live_sums, spectrum, (const int *)wide_flag,
                                                       (const int *)mk.scan_stamp, mk.stamp);
        GBFG_LAUNCH_CHECK("scan_add_kernel");
        return GBFG_OK;
    } else {
        scan_tile_sums_kernel<<<grid, SCAN_THREADS, 0, st>>>(diff, n_bins, tiles, tile_sums, wide_flag, mk.scan_stamp, mk.stamp);
        GBFG_LAUNCH_CHECK("scan_tile_sums_kernel");
    }
    cudaError_t e = launch_dependent(scan_add_kernel, grid, dim3(SCAN_THREADS), 0, st, diff, n_bins, tiles,
                                     (const int64_t *)tile_sums, spectrum, (const int *)wide_flag, (const int *)mk.scan_stamp, mk.stamp);
    if (e != cudaSuccess) return set_cuda_error(e, "scan_add_kernel");
    GBFG_LAUNCH_CHECK("scan_add_kernel");
    return GBFG_OK;
}

}  // namespace gbfg
