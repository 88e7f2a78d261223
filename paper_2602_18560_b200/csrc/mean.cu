// mean.cu — the running-mean estimator of eq. (D1) (the paper's production choice,
// :176, :552), R8: window sums over W = 2h+1 bins centred on k, ends reflected, fused with
//     psd[k] = s_instr[k] + (sum[k] * 2^scale_log2) / W          (eq. 10).
//
// This stage IS bound by HBM: 32 bytes per bin (spectrum in, sum out, s_instr in, PSD out) against a
// few integer additions.  One CTA stages a tile of outputs and its two h-bin halos in shared memory,
// turns it into an inclusive prefix sum in place (every warp scans a contiguous segment, 32 bins per
// step, then the segment totals are scanned), and writes sum[k] = P[k + 2h] - P[k - 1] coalesced.
// The halos are re-read through L2, not HBM.  Integer arithmetic: exact, any order.
#include "gbfg_common.cuh"

namespace gbfg {

#ifndef MEAN_CFG_THREADS
#define MEAN_CFG_THREADS 512
#define MEAN_CFG_LT 8192      /* 64 KB of int64 per CTA, three CTAs per SM: the best of the sweep in profiles/r01_mean_kernel.md */
#define MEAN_CFG_CTAS 3
#endif
constexpr int MEAN_THREADS = MEAN_CFG_THREADS;
constexpr int MEAN_WARPS = MEAN_THREADS / 32;
constexpr int MEAN_LT = MEAN_CFG_LT;            // positions per tile, halos included
constexpr int MEAN_CTAS = MEAN_CFG_CTAS;        // CTAs per SM
constexpr int MEAN_SEG = MEAN_LT / MEAN_WARPS; // 768 positions per warp
constexpr size_t MEAN_SMEM = sizeof(int64_t) * MEAN_LT;
constexpr int MEAN_STAGE_UNROLL = 8;           // positions per thread = LT / THREADS, in batches of eight loads
constexpr int MEAN_OUT_UNROLL = 4;

struct MeanArgs {
    const int64_t *x;        // [n_cat][n]
    int64_t *sum;            // [n_cat][n]
    const double *s_instr;   // [n] or NULL (no PSD)
    double *psd;             // [n_cat][n] or NULL
    int *neg_flag;           // nullable: set to 1 when a window sum is negative
    unsigned long long *delta_bits;   // nullable: [n_cat] largest relative PSD change of the row, as binary64 bits (R13)
    const int *cum;          // nullable: [n_cat][n_dblk + 1] dirty blocks before each block (DirtyView); a tile without one is skipped
    int n_dblk, dblk_log2;
    int64_t n;
    int h;
    int S;                   // outputs per tile
    double scale, w;         // 2^scale_log2 and (double)W
};

__global__ void __launch_bounds__(MEAN_THREADS, MEAN_CTAS)
running_mean_kernel(MeanArgs a)
{
    extern __shared__ __align__(16) unsigned char mean_smem[];
    int64_t *P = reinterpret_cast<int64_t *>(mean_smem);
    __shared__ int64_t seg_off[MEAN_WARPS];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int64_t row = (int64_t)blockIdx.y * a.n;
    const int64_t o0 = (int64_t)blockIdx.x * a.S;
    const int n_out = (int)((a.n - o0 < a.S) ? (a.n - o0) : a.S);
    if (a.cum) {                                           // no output of the tile saw a changed bin: sums and PSD stand
        const int *cum = a.cum + (int64_t)blockIdx.y * (a.n_dblk + 1);
        if (cum[((o0 + n_out - 1) >> a.dblk_log2) + 1] == cum[o0 >> a.dblk_log2]) return;
    }
    const int h = a.h;
    const int Lt = n_out + 2 * h;                          // position p <-> bin o0 - h + p, reflected

    // stage: MEAN_STAGE_UNROLL independent loads in flight per thread (the kernel lives on memory-level parallelism)
    for (int p0 = tid; p0 < MEAN_LT; p0 += MEAN_STAGE_UNROLL * MEAN_THREADS) {
        int64_t v[MEAN_STAGE_UNROLL];
#pragma unroll
        for (int u = 0; u < MEAN_STAGE_UNROLL; ++u) {
            const int p = p0 + u * MEAN_THREADS;
            v[u] = 0;
            if (p < Lt) {
                int64_t g = o0 - h + p;
                if (g < 0) g = -g - 1;
                if (g >= a.n) g = 2 * a.n - 1 - g;
                v[u] = __ldg(a.x + row + g);
            }
        }
#pragma unroll
        for (int u = 0; u < MEAN_STAGE_UNROLL; ++u)
            if (p0 + u * MEAN_THREADS < MEAN_LT) P[p0 + u * MEAN_THREADS] = v[u];
    }
    __syncthreads();
    // inclusive scan of the warp's segment, 32 consecutive positions per step
    {
        int64_t carry = 0;
        const int base = warp * MEAN_SEG;
        for (int q = 0; q < MEAN_SEG; q += 32) {
            int64_t v = P[base + q + lane];
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const int64_t up = __shfl_up_sync(0xffffffffu, v, o);
                if (lane >= o) v += up;
            }
            v += carry;
            P[base + q + lane] = v;
            carry = __shfl_sync(0xffffffffu, v, 31);
        }
        if (lane == 0) seg_off[warp] = carry;             // segment total
    }
    __syncthreads();
    if (warp == 0) {                                       // exclusive scan of the segment totals
        int64_t v = lane < MEAN_WARPS ? seg_off[lane] : 0;
        const int64_t own = v;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int64_t up = __shfl_up_sync(0xffffffffu, v, o);
            if (lane >= o) v += up;
        }
        if (lane < MEAN_WARPS) seg_off[lane] = v - own;
    }
    __syncthreads();
    bool neg = false;
    double dmax = 0.0;
    for (int j0 = tid; j0 < n_out; j0 += MEAN_OUT_UNROLL * MEAN_THREADS) {
        double si[MEAN_OUT_UNROLL];
        if (a.psd) {
#pragma unroll
            for (int u = 0; u < MEAN_OUT_UNROLL; ++u) {
                const int j = j0 + u * MEAN_THREADS;
                si[u] = j < n_out ? __ldg(a.s_instr + o0 + j) : 0.0;
            }
        }
#pragma unroll
        for (int u = 0; u < MEAN_OUT_UNROLL; ++u) {
            const int j = j0 + u * MEAN_THREADS;
            if (j < n_out) {
                const int hi = j + 2 * h;                  // window of output j = positions [j, j + 2h]
                int64_t sv = P[hi] + seg_off[hi / MEAN_SEG];
                if (j > 0) sv -= P[j - 1] + seg_off[(j - 1) / MEAN_SEG];
                const int64_t g = o0 + j;
                a.sum[row + g] = sv;
                neg |= sv < 0;
                if (a.psd) {
                    const double e = (double)sv * a.scale;
                    const double m = e / a.w;
                    const double pnew = si[u] + m;
                    if (a.delta_bits) {
                        const double pold = a.psd[row + g];
                        const double d = fabs(pnew - pold) / pold;
                        if (d > dmax) dmax = d;
                    }
                    a.psd[row + g] = pnew;
                }
            }
        }
    }
    if (a.delta_bits) {
        for (int o = 16; o; o >>= 1) dmax = fmax(dmax, __shfl_xor_sync(0xffffffffu, dmax, o));
        if (lane == 0 && dmax > 0.0) atomicMax(a.delta_bits + blockIdx.y, (unsigned long long)__double_as_longlong(dmax));
    }
    if (a.neg_flag && neg) *a.neg_flag = 1;
}

// internal entry: window sums (+ PSD when psd != NULL) of every row
int launch_mean(const DirtyView *dv, const int64_t *x, int64_t n_bins, int n_cat, int window, int64_t *sum,
                const double *s_instr, double *psd, int scale_log2, int *neg_flag, unsigned long long *delta_bits,
                cudaStream_t st)
{
    MeanArgs a;
    a.cum = dv ? dv->cum : nullptr;
    a.n_dblk = dv ? dv->n_dblk : 0;
    a.dblk_log2 = dv ? dv->dblk_log2 : 0;
    a.delta_bits = delta_bits;
    a.x = x; a.sum = sum; a.s_instr = s_instr; a.psd = psd; a.neg_flag = neg_flag;
    a.n = n_bins; a.h = window / 2;
    const int s_max = MEAN_LT - (window - 1);
    const int slots = MEAN_CTAS * sm_count();
    int64_t tiles = (n_bins + s_max - 1) / s_max;
    if (tiles * n_cat > slots && n_cat == 1) tiles = (tiles + slots - 1) / slots * slots;   // whole waves of CTAs
    a.S = (int)((n_bins + tiles - 1) / tiles);
    tiles = (n_bins + a.S - 1) / a.S;
    a.scale = ldexp(1.0, scale_log2);
    a.w = (double)window;
    static thread_local int attr_dev = -1;
    int dev = 0;
    GBFG_CUDA(cudaGetDevice(&dev));
    if (attr_dev != dev) {
        GBFG_CUDA(cudaFuncSetAttribute(running_mean_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)MEAN_SMEM));
        attr_dev = dev;
    }
    {
        LaunchTimer lt(K_MEDIAN, st);
        running_mean_kernel<<<dim3((unsigned)tiles, (unsigned)n_cat), MEAN_THREADS, MEAN_SMEM, st>>>(a);
    }
    GBFG_LAUNCH_CHECK("running_mean_kernel");
    return GBFG_OK;
}

}  // namespace gbfg

using namespace gbfg;

extern "C" int gbfg_running_mean(const int64_t *dev_spectrum, int64_t n_bins, int32_t n_cat, int32_t window,
                                 int64_t *dev_sum_out, const double *dev_s_instr, int32_t scale_log2,
                                 double *dev_psd, void *stream)
{
    if (!dev_spectrum || !dev_sum_out || dev_spectrum == dev_sum_out) return GBFG_ERR_INVALID_ARG;
    if (window < 1 || (window & 1) == 0 || n_cat < 1 || n_bins < 1 || n_bins >= 2147483648ll) return GBFG_ERR_INVALID_ARG;
    if ((dev_psd != nullptr) != (dev_s_instr != nullptr)) return GBFG_ERR_INVALID_ARG;
    if (scale_log2 < -1000 || scale_log2 > 0) return GBFG_ERR_INVALID_ARG;
    if (window > GBFG_MAX_WINDOW || n_cat > GBFG_MAX_CAT) return GBFG_ERR_UNSUPPORTED;
    if (n_bins < window / 2 + 1) return GBFG_ERR_INVALID_ARG;
    int rc = check_device();
    if (rc) return rc;
    return launch_mean(nullptr, dev_spectrum, n_bins, n_cat, window, dev_sum_out, dev_s_instr, dev_psd, scale_log2, nullptr, nullptr,
                       (cudaStream_t)stream);
}
