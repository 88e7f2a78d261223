// median.cu — stage (iii): exact running median of eq. (D2) + the PSD of eq. (10).
//
// DESIGN.md R3: odd window W = 2h+1 centred on k, ends reflected, statistic = the h-th smallest
// of the 2h+1 int64 values.  Only integer comparisons decide the result, so it is exact.
//
// One CTA per tile of S = LT - 2h outputs.  The tile and its two h-bin halos (LT positions) are
// staged in shared memory and sorted ONCE by (value, position).  With the sorted order in hand a
// window is a position interval, and its median is found without ever sorting a window:
//   * a (rank-bucket x position-block) table of counts locates, by bisection, the h-th smallest
//     element of a block-aligned position interval (start of a chunk of 32 outputs);
//   * from there one thread walks its chunk: sliding the window by one bin removes one position
//     and adds one, which moves the median by at most one place in the sorted order; the
//     neighbouring in-window element is found by stepping through the sorted positions
//     (on average LT/W steps).
// The per-output rank is kept in shared memory and written out coalesced, fused with
//     psd[k] = s_instr[k] + C * (med[k] * 2^scale_log2)        (eqs. 10, D2, D3).
#include "gbfg_common.cuh"

namespace gbfg {

constexpr int MED_LT = 8192;                  // positions per tile, halos included (power of two)
constexpr int MED_THREADS = 1024;
constexpr int MED_PB = 32;                    // position block = outputs per chunk
constexpr int MED_RB = 128;                   // sorted ranks per bucket
constexpr int MED_NPB = MED_LT / MED_PB;      // 256
constexpr int MED_NRB = MED_LT / MED_RB;      // 64
constexpr int MED_TROW = MED_NPB + 2;         // table row stride in u16 (even: rows stay 4-byte aligned)
constexpr uint64_t SIGN64 = 0x8000000000000000ull;

constexpr size_t MED_SMEM = sizeof(uint64_t) * MED_LT      // skey
                          + sizeof(uint16_t) * MED_LT      // spos
                          + sizeof(uint16_t) * MED_LT      // rop
                          + sizeof(uint16_t) * MED_LT      // orank
                          + sizeof(uint16_t) * MED_NRB * MED_TROW;

struct MedianArgs {
    const int64_t *x;        // [n_cat][n]
    int64_t *med;            // [n_cat][n]
    const double *s_instr;   // [n] or NULL (no PSD)
    double *psd;             // [n_cat][n] or NULL
    const uint8_t *tile_dirty; // [n_cat][tiles] or NULL: skip tiles whose flag is 0
    int64_t n;
    int h;
    int S;                   // outputs per tile = MED_LT - 2h
    int tiles;
    double norm, scale;      // C and 2^scale_log2
};

__global__ void __launch_bounds__(MED_THREADS, 1)
running_median_kernel(MedianArgs a)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    uint64_t *skey = reinterpret_cast<uint64_t *>(smem_raw);
    uint16_t *spos = reinterpret_cast<uint16_t *>(skey + MED_LT);
    uint16_t *rop = spos + MED_LT;
    uint16_t *orank = rop + MED_LT;
    uint16_t *tab = orank + MED_LT;
    uint32_t *tab32 = reinterpret_cast<uint32_t *>(tab);

    const int tid = threadIdx.x;
    const int tile = blockIdx.x;
    if (a.tile_dirty && a.tile_dirty[(int64_t)blockIdx.y * a.tiles + tile] == 0) return;
    const int64_t row = (int64_t)blockIdx.y * a.n;
    const int64_t o0 = (int64_t)tile * a.S;
    const int h = a.h, W = 2 * a.h + 1;
    const int n_out = (int)((a.n - o0 < a.S) ? (a.n - o0) : a.S);
    const int Lt = n_out + 2 * h;                        // positions really used

    // ---- stage the tile: position p <-> global bin o0 - h + p, reflected at both ends
    for (int p = tid; p < MED_LT; p += MED_THREADS) {
        uint64_t key = ~0ull;
        if (p < Lt) {
            int64_t g = o0 - h + p;
            if (g < 0) g = -g - 1;
            if (g >= a.n) g = 2 * a.n - 1 - g;
            key = (uint64_t)a.x[row + g] ^ SIGN64;
        }
        skey[p] = key;
        spos[p] = (uint16_t)p;
    }
    for (int e = tid; e < MED_NRB * MED_TROW / 2; e += MED_THREADS) tab32[e] = 0u;
    __syncthreads();

    // ---- bitonic sort by (key, position)
    for (int k = 2; k <= MED_LT; k <<= 1) {
        for (int j = k >> 1; j > 0; j >>= 1) {
            for (int t = tid; t < MED_LT / 2; t += MED_THREADS) {
                int i = ((t & ~(j - 1)) << 1) | (t & (j - 1));
                int l = i | j;
                bool up = (i & k) == 0;
                uint64_t ka = skey[i], kb = skey[l];
                uint16_t pa = spos[i], pb = spos[l];
                bool gt = (ka > kb) || (ka == kb && pa > pb);
                if (gt == up) { skey[i] = kb; skey[l] = ka; spos[i] = pb; spos[l] = pa; }
            }
            __syncthreads();
        }
    }

    // ---- inverse permutation and the count table
    for (int r = tid; r < MED_LT; r += MED_THREADS) {
        int p = spos[r];
        rop[p] = (uint16_t)r;
        int e = (r / MED_RB) * MED_TROW + (p / MED_PB) + 1;
        atomicAdd(&tab32[e >> 1], (e & 1) ? 0x10000u : 1u);
    }
    __syncthreads();
    // prefix along the position blocks: tab[rb][pb] = #{r in bucket rb : pos < pb*PB}
    {
        const int warp = tid >> 5, lane = tid & 31;
        constexpr int PER = (MED_NPB + 1 + 31) / 32;     // 9 entries per lane
        for (int rb = warp; rb < MED_NRB; rb += MED_THREADS / 32) {
            uint16_t *rowp = tab + rb * MED_TROW;
            int v[PER], s = 0;
#pragma unroll
            for (int q = 0; q < PER; ++q) {
                int idx = lane * PER + q;
                v[q] = idx <= MED_NPB ? rowp[idx] : 0;
                s += v[q];
            }
            int incl = s;
            for (int o = 1; o < 32; o <<= 1) {
                int up = __shfl_up_sync(0xffffffffu, incl, o);
                if (lane >= o) incl += up;
            }
            int run = incl - s;
#pragma unroll
            for (int q = 0; q < PER; ++q) {
                int idx = lane * PER + q;
                run += v[q];
                if (idx <= MED_NPB) rowp[idx] = (uint16_t)run;
            }
        }
    }
    __syncthreads();
    // exclusive prefix along the rank buckets: tab[rb][pb] = #{r < rb*RB : pos < pb*PB}
    for (int pb = tid; pb <= MED_NPB; pb += MED_THREADS) {
        int run = 0;
        for (int rb = 0; rb < MED_NRB; ++rb) {
            int v = tab[rb * MED_TROW + pb];
            tab[rb * MED_TROW + pb] = (uint16_t)run;
            run += v;
        }
    }
    __syncthreads();

    // ---- one thread per chunk of PB outputs
    const int n_chunks = (n_out + MED_PB - 1) / MED_PB;
    if (tid < n_chunks) {
        const int j0 = tid * MED_PB;
        const int j1 = (j0 + MED_PB < n_out) ? j0 + MED_PB : n_out;
        const int b0 = tid, b1 = (j0 + W) / MED_PB;
        const int na = b1 * MED_PB - j0;
        int plo = j0, phi, m, below;
        if (na > 0) {
            const int t = (h < na - 1) ? h : na - 1;
            int lo = 0, hi = MED_NRB;
            while (hi - lo > 1) {
                int mid = (lo + hi) >> 1;
                int cnt = (int)tab[mid * MED_TROW + b1] - (int)tab[mid * MED_TROW + b0];
                if (cnt <= t) lo = mid; else hi = mid;
            }
            int need = t - ((int)tab[lo * MED_TROW + b1] - (int)tab[lo * MED_TROW + b0]);
            const unsigned span = (unsigned)(na - 1);
            m = lo * MED_RB;
            for (;; ++m) {
                if ((unsigned)((int)spos[m] - j0) <= span) {
                    if (need == 0) break;
                    --need;
                }
            }
            below = t;
            phi = b1 * MED_PB - 1;
        } else {
            m = MED_LT; below = 0; phi = j0 - 1;
        }
#define IN_SET(r) ((unsigned)((int)spos[r] - plo) <= (unsigned)(phi - plo))
#define REBALANCE()                                                                  \
        do {                                                                         \
            while (below > h) { do { --m; } while (!IN_SET(m)); --below; }           \
            while (below < h && m < MED_LT) {                                        \
                do { ++m; } while (m < MED_LT && !IN_SET(m));                        \
                ++below;                                                             \
            }                                                                        \
        } while (0)
        for (int p = phi + 1; p < j0 + W; ++p) {         // complete the first window
            phi = p;
            if ((int)rop[p] < m) ++below;
        }
        REBALANCE();
        orank[j0] = (uint16_t)m;
        for (int j = j0 + 1; j < j1; ++j) {
            int gone = rop[plo];                          // position j-1 leaves
            ++plo;
            int come = rop[phi + 1];                      // position j+2h enters
            ++phi;
            if (gone < m) --below;
            else if (gone == m) { do { ++m; } while (m < MED_LT && !IN_SET(m)); }
            if (come < m) ++below;
            REBALANCE();
            orank[j] = (uint16_t)m;
        }
#undef IN_SET
#undef REBALANCE
    }
    __syncthreads();

    // ---- coalesced epilogue: median and PSD
    for (int j = tid; j < n_out; j += MED_THREADS) {
        int64_t v = (int64_t)(skey[orank[j]] ^ SIGN64);
        int64_t g = o0 + j;
        a.med[row + g] = v;
        if (a.psd) {
            double e = (double)v * a.scale;
            a.psd[row + g] = a.s_instr[g] + a.norm * e;
        }
    }
}

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

int median_tiles(int64_t n_bins, int window)
{
    int S = MED_LT - (window - 1);
    return (int)((n_bins + S - 1) / S);
}

// internal entry: median (+ PSD when psd != NULL) of every row; tile_dirty nullable
int launch_median(const int64_t *x, int64_t n_bins, int n_cat, int window, int64_t *med,
                  const double *s_instr, double *psd, double norm, int scale_log2,
                  const uint8_t *tile_dirty, cudaStream_t st)
{
    MedianArgs a;
    a.x = x; a.med = med; a.s_instr = s_instr; a.psd = psd; a.tile_dirty = tile_dirty;
    a.n = n_bins; a.h = window / 2; a.S = MED_LT - 2 * a.h;
    a.tiles = median_tiles(n_bins, window);
    a.norm = norm; a.scale = ldexp(1.0, scale_log2);
    static thread_local int attr_dev = -1;
    int dev = 0;
    GBFG_CUDA(cudaGetDevice(&dev));
    if (attr_dev != dev) {
        GBFG_CUDA(cudaFuncSetAttribute(running_median_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)MED_SMEM));
        attr_dev = dev;
    }
    dim3 grid(a.tiles, n_cat);
    {
        LaunchTimer lt(K_MEDIAN, st);
        running_median_kernel<<<grid, MED_THREADS, MED_SMEM, st>>>(a);
    }
    GBFG_LAUNCH_CHECK("running_median_kernel");
    return GBFG_OK;
}

}  // namespace gbfg

using namespace gbfg;

extern "C" int gbfg_running_median(const int64_t *dev_spectrum, int64_t n_bins, int32_t n_cat, int32_t window,
                                   int64_t *dev_median_out, void *stream)
{
    if (!dev_spectrum || !dev_median_out || dev_spectrum == dev_median_out) return GBFG_ERR_INVALID_ARG;
    if (window < 1 || (window & 1) == 0 || n_cat < 1 || n_bins < 1 || n_bins >= 2147483648ll) return GBFG_ERR_INVALID_ARG;
    if (window > GBFG_MAX_WINDOW || n_cat > GBFG_MAX_CAT) return GBFG_ERR_UNSUPPORTED;
    if (n_bins < window / 2 + 1) return GBFG_ERR_INVALID_ARG;
    int rc = check_device();
    if (rc) return rc;
    return launch_median(dev_spectrum, n_bins, n_cat, window, dev_median_out, nullptr, nullptr, 1.0, 0, nullptr,
                         (cudaStream_t)stream);
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
