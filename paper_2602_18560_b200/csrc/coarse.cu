// coarse.cu — coarse-graining of the PSD, eqs. (13)-(14), and the characteristic
// strain of eq. (B1); R10.  The epilogue that turns the ~4e6-bin PSD of one
// catalog into the ~100 numbers the inference uses.
//
// One CTA per (coarse bin, row).  The mean of a coarse bin is a sum of up to ~1e5 positive binary64
// terms: every thread adds its stride of the bin with a compensated (Kahan) sum, the 256 partial sums
// are combined by a tree, so the result is within a few ulp of the exactly rounded sum the oracle
// forms (math.fsum); the test tolerance is 1e-14 relative.  The mean frequency of eq. (14) is the
// mean of an arithmetic progression of bin centres: closed form, no sum.
#include "gbfg_common.cuh"

namespace gbfg {

constexpr int COARSE_THREADS = 256;

__global__ void __launch_bounds__(COARSE_THREADS)
coarse_grain_kernel(const double *__restrict__ psd, int64_t n_bins, const int64_t *__restrict__ edges,
                    double f_min, double t_obs, double *__restrict__ S, double *__restrict__ fk,
                    double *__restrict__ hc)
{
    __shared__ double part[COARSE_THREADS];
    const int k = blockIdx.x, n_coarse = gridDim.x;
    const int64_t row = (int64_t)blockIdx.y * n_bins;
    int64_t i0 = edges[k], i1 = edges[k + 1];
    if (i0 < 0) i0 = 0;
    if (i1 > n_bins) i1 = n_bins;
    const int64_t nk = i1 - i0;
    double sum = 0.0, comp = 0.0;                          // Kahan: sum + comp carries the rounding errors
    for (int64_t i = i0 + threadIdx.x; i < i1; i += COARSE_THREADS) {
        const double y = psd[row + i] - comp;
        const double t = sum + y;
        comp = (t - sum) - y;
        sum = t;
    }
    part[threadIdx.x] = sum;
    __syncthreads();
    for (int s = COARSE_THREADS / 2; s > 0; s >>= 1) {
        if ((int)threadIdx.x < s) part[threadIdx.x] = part[threadIdx.x] + part[threadIdx.x + s];
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        const double nan = __longlong_as_double(0x7ff8000000000000ll);
        double mean_s = nan, mean_f = nan;
        if (nk > 0) {
            mean_s = part[0] / (double)nk;
            // mean of f_min + (i + 1/2)/T over i0 <= i < i1
            mean_f = f_min + (0.5 * (double)(i0 + i1 - 1) + 0.5) / t_obs;
        }
        S[(int64_t)blockIdx.y * n_coarse + k] = mean_s;
        if (blockIdx.y == 0 && fk) fk[k] = mean_f;
        if (hc) hc[(int64_t)blockIdx.y * n_coarse + k] = sqrt(mean_f * mean_s);
    }
}

}  // namespace gbfg

using namespace gbfg;

extern "C" int gbfg_coarse_grain(const double *dev_psd, int64_t n_bins, int32_t n_cat, const int64_t *dev_edges,
                                 int32_t n_coarse, double f_min, double t_obs, double *dev_S, double *dev_f,
                                 double *dev_hc, void *stream)
{
    if (!dev_psd || !dev_edges || !dev_S) return GBFG_ERR_INVALID_ARG;
    if (n_bins < 1 || n_cat < 1 || n_coarse < 1 || n_coarse > 65535 || !(f_min > 0.0) || !(t_obs > 0.0)) return GBFG_ERR_INVALID_ARG;
    if (n_cat > GBFG_MAX_CAT) return GBFG_ERR_UNSUPPORTED;
    int rc = check_device();
    if (rc) return rc;
    {
        LaunchTimer lt(K_PSD, (cudaStream_t)stream);
        coarse_grain_kernel<<<dim3((unsigned)n_coarse, (unsigned)n_cat), COARSE_THREADS, 0, (cudaStream_t)stream>>>(
            dev_psd, n_bins, dev_edges, f_min, t_obs, dev_S, dev_f, dev_hc);
    }
    GBFG_LAUNCH_CHECK("coarse_grain_kernel");
    return GBFG_OK;
}
