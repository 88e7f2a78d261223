// snr.cu — stage (iv): rho^2 of every unresolved source against the current PSD, threshold test
// and compaction of the newly resolved (eqs. 11-12; R4).
//
//   rho2_i = sum_{k = k0 .. k0 + w_eff - 1} (4 p_i) / psd[k]
//
// Narrow sources (w_eff <= SNR_NARROW, ~90 % of a catalog) are summed by their own thread in
// ascending k with one division per bin: bit-identical to the definition.  Wider chirps (up to
// 7e4 bins at 4 yr) are summed by the whole warp over 1/psd, using per-256-bin block sums of
// 1/psd for the interior, then multiplied by 4p: relative difference from the ascending sum is a few 1e-16
// per term, far inside the 1e-12 contract.  A source whose rho2 lands within 1e-9 (relative) of
// the threshold is re-summed in ascending order with the definition's arithmetic, so the
// resolved/unresolved decision is always taken on the definition's value.
// Selection: warp ballot + one atomic per warp reserves slots in the index list.
#include "gbfg_common.cuh"

namespace gbfg {

constexpr int SNR_NARROW = 8;
constexpr int SNR_IB = 256;          // bins per block sum of 1/psd

// inv_blocks[c][j] = sum_{k in [256 j, 256 j + 256)} 1 / psd[c][k]   (fixed tree order)
__global__ void __launch_bounds__(256)
inv_block_sums_kernel(const double *__restrict__ psd, int64_t n_bins, int blocks_per_row,
                      double *__restrict__ inv_blocks)
{
    __shared__ double wsum[8];
    const int64_t row = (int64_t)blockIdx.y * n_bins;
    for (int jb = blockIdx.x; jb < blocks_per_row; jb += gridDim.x) {
        int64_t k = (int64_t)jb * SNR_IB + threadIdx.x;
        double v = k < n_bins ? 1.0 / psd[row + k] : 0.0;
        for (int o = 16; o; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        if ((threadIdx.x & 31) == 0) wsum[threadIdx.x >> 5] = v;
        __syncthreads();
        if (threadIdx.x == 0) {
            double s = ((wsum[0] + wsum[1]) + (wsum[2] + wsum[3])) + ((wsum[4] + wsum[5]) + (wsum[6] + wsum[7]));
            inv_blocks[(int64_t)blockIdx.y * blocks_per_row + jb] = s;
        }
        __syncthreads();
    }
}

__device__ __forceinline__ double warp_sum(double v)
{
    for (int o = 16; o; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// sum over [k0, k1) of 1/psd, all 32 lanes cooperate (arguments warp-uniform)
__device__ __forceinline__ double warp_inv_sum(const double *__restrict__ psd_row, const double *__restrict__ ib_row,
                                               int64_t k0, int64_t k1, int lane)
{
    double acc = 0.0;
    int64_t jb0 = (k0 + SNR_IB - 1) / SNR_IB, jb1 = k1 / SNR_IB;
    if (ib_row && jb1 > jb0) {
        for (int64_t k = k0 + lane; k < jb0 * SNR_IB; k += 32) acc += 1.0 / psd_row[k];
        for (int64_t j = jb0 + lane; j < jb1; j += 32) acc += ib_row[j];
        for (int64_t k = jb1 * SNR_IB + lane; k < k1; k += 32) acc += 1.0 / psd_row[k];
    } else {
        for (int64_t k = k0 + lane; k < k1; k += 32) acc += 1.0 / psd_row[k];
    }
    return warp_sum(acc);
}

struct SnrArgs {
    const double *A, *f, *fdot;
    const double *psd;          // [n_cat][n_bins]
    const double *inv_blocks;   // [n_cat][blocks_per_row] or NULL
    int blocks_per_row;
    const int64_t *cand_idx;    // NULL = every source; else a list of global indices ...
    const int64_t *cand_count;  // ... with its length on the device
    int64_t n_all;
    double thr;                 // rho_th^2
    uint8_t *resolved;
    double *rho2_out;           // nullable
    int64_t *sel_idx;
    int64_t *sel_count;         // [1 + n_cat]
    int64_t *near_count;        // nullable; one counter, or one per catalog
    int near_per_cat;
};

__global__ void __launch_bounds__(256)
snr_select_kernel(GridDev g, CatTable ct, SnrArgs a)
{
    const int lane = threadIdx.x & 31;
    const int64_t n = a.cand_idx ? *a.cand_count : a.n_all;
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    // whole warps iterate together (the loop bound is rounded up to a warp)
    const int64_t n_round = (n + 31) & ~(int64_t)31;
    for (int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; t < n_round; t += stride) {
        int64_t i = -1;
        bool test = false;
        if (t < n) {
            i = a.cand_idx ? a.cand_idx[t] : t;
            test = a.resolved[i] == 0;
        }
        SrcBins s; s.status = 1; s.k0 = 0; s.w_eff = 0; s.p = 0.0; s.q = 0;
        int cat = 0;
        if (test) {
            s = source_bins(g, a.A[i], a.f[i], a.fdot[i]);
            cat = cat_of(ct, i);
        }
        const bool ok = test && s.status == 0;
        const double four_p = 4.0 * s.p;
        const double *psd_row = a.psd + (int64_t)cat * g.n_bins;
        double r2 = 0.0;
        if (ok && s.w_eff <= SNR_NARROW) {
            for (int64_t k = s.k0; k < s.k0 + s.w_eff; ++k) r2 = r2 + four_p / psd_row[k];
        }
        // wide sources: one at a time, the whole warp sums
        unsigned wide = __ballot_sync(0xffffffffu, ok && s.w_eff > SNR_NARROW);
        while (wide) {
            const int src = __ffs(wide) - 1;
            wide &= wide - 1;
            const int64_t k0 = __shfl_sync(0xffffffffu, s.k0, src);
            const int64_t we = __shfl_sync(0xffffffffu, s.w_eff, src);
            const int c = __shfl_sync(0xffffffffu, cat, src);
            const double *pr = a.psd + (int64_t)c * g.n_bins;
            const double *ir = a.inv_blocks ? a.inv_blocks + (int64_t)c * a.blocks_per_row : nullptr;
            double tot = warp_inv_sum(pr, ir, k0, k0 + we, lane);
            if (lane == src) r2 = four_p * tot;
        }
        bool sel = false, near = false;
        if (ok) {
            if (fabs(r2 / a.thr - 1.0) <= 4e-9 && s.w_eff > SNR_NARROW) {
                // decision on the definition's ascending sum
                double acc = 0.0;
                for (int64_t k = s.k0; k < s.k0 + s.w_eff; ++k) acc = acc + four_p / psd_row[k];
                r2 = acc;
            }
            near = fabs(r2 / a.thr - 1.0) <= 2e-9;
            sel = r2 > a.thr;
        }
        if (test && a.rho2_out) a.rho2_out[i] = ok ? r2 : __longlong_as_double(0x7ff8000000000000ll);
        const unsigned sel_mask = __ballot_sync(0xffffffffu, sel);
        const unsigned near_mask = __ballot_sync(0xffffffffu, near);
        if (sel_mask) {
            int64_t base = 0;
            if (lane == 0) base = (int64_t)atomicAdd((unsigned long long *)a.sel_count, (unsigned long long)__popc(sel_mask));
            base = __shfl_sync(0xffffffffu, base, 0);
            if (sel) {
                a.sel_idx[base + __popc(sel_mask & ((1u << lane) - 1u))] = i;
                a.resolved[i] = 1;
                atomicAdd((unsigned long long *)(a.sel_count + 1 + cat), 1ull);
            }
        }
        if (near_mask && a.near_count) {
            if (a.near_per_cat) { if (near) atomicAdd((unsigned long long *)(a.near_count + cat), 1ull); }
            else if (lane == 0) atomicAdd((unsigned long long *)a.near_count, (unsigned long long)__popc(near_mask));
        }
    }
}

int snr_inv_blocks_per_row(int64_t n_bins) { return (int)((n_bins + SNR_IB - 1) / SNR_IB); }

// internal entry.  inv_blocks: scratch [n_cat * blocks_per_row] doubles (or NULL: direct sums only).
// sel_count[0 .. n_cat] must be zero on entry.
int launch_snr_select(const GridDev &g, const CatTable &ct, const double *A, const double *f, const double *fdot,
                      const double *psd, double rho_th, uint8_t *resolved, double *rho2_out,
                      const int64_t *cand_idx, const int64_t *cand_count, int64_t n_launch,
                      int64_t *sel_idx, int64_t *sel_count, int64_t *near_count, int near_per_cat,
                      double *inv_blocks, cudaStream_t st)
{
    const int bpr = snr_inv_blocks_per_row(g.n_bins);
    if (inv_blocks) {
        int bx = bpr < sm_count() * 8 ? bpr : sm_count() * 8;
        {
            LaunchTimer lt(K_INV_BLOCKS, st);
            inv_block_sums_kernel<<<dim3(bx, ct.n_cat), 256, 0, st>>>(psd, g.n_bins, bpr, inv_blocks);
        }
        GBFG_LAUNCH_CHECK("inv_block_sums_kernel");
    }
    if (n_launch <= 0) return GBFG_OK;
    SnrArgs a;
    a.A = A; a.f = f; a.fdot = fdot; a.psd = psd; a.inv_blocks = inv_blocks; a.blocks_per_row = bpr;
    a.cand_idx = cand_idx; a.cand_count = cand_count; a.n_all = ct.offsets[ct.n_cat];
    a.thr = rho_th * rho_th;
    a.resolved = resolved; a.rho2_out = rho2_out; a.sel_idx = sel_idx; a.sel_count = sel_count;
    a.near_count = near_count; a.near_per_cat = near_per_cat;
    int64_t blocks = (n_launch + 255) / 256;
    int64_t cap = (int64_t)sm_count() * 16;
    if (blocks > cap) blocks = cap;
    {
        LaunchTimer lt(K_SNR, st);
        snr_select_kernel<<<(int)blocks, 256, 0, st>>>(g, ct, a);
    }
    GBFG_LAUNCH_CHECK("snr_select_kernel");
    return GBFG_OK;
}

}  // namespace gbfg
