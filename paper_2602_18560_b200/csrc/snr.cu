// snr.cu — stage (iv): rho^2 of every unresolved source against the current PSD, threshold test
// and compaction of the newly resolved (eqs. 11-12; R4, R5).
//
//   rho2_i = sum_{k = k0 .. k0 + w_eff - 1} (4 p_i) / psd[k]
//
// Three pieces:
//  * candidate records (cand_build_kernel).  One pass over the catalog keeps, for every source that
//    can still be resolved, its first bin, width, 4p and index.  With pre-selection (R5;
//    steps 2-3 of the algorithm) a source is kept only if its rho^2 against the
//    instrument noise alone reaches the threshold: S_n >= S_instr, so nothing else ever can.
//  * an exact prefix of 1/psd (inv_prefix kernels).  1/psd[k] is rounded once (IEEE division) and
//    accumulated as a 128-bit fixed-point integer, so sum_{k0 <= k < k1} 1/psd[k] is a difference of
//    two prefixes, exact and independent of the order of accumulation.  (A binary64 prefix is not
//    accurate enough: its differences are off by up to 2e-10.)
//  * the test (snr_cand_kernel), one thread per candidate.  Narrow sources (w_eff <= SNR_NARROW) are
//    summed in ascending k with one division per bin: bit-identical to the definition.  Wider chirps
//    (up to 7e4 bins at 4 yr) take 4p * (prefix difference): relative difference from the ascending
//    sum is a few 1e-16 per term, far inside the 1e-12 contract.  A source whose rho2 lands within
//    4e-9 (relative) of the threshold is re-summed in ascending order with the definition's
//    arithmetic, so the resolved/unresolved decision is always taken on the definition's value.
//    Selection: warp ballot + one atomic per warp reserves slots in the index list.
#include "gbfg_common.cuh"

namespace gbfg {

constexpr int SNR_NARROW = 4;
constexpr int SNR_SEL_CAP = 1024;              // selected indices a CTA holds before it appends them to the list
constexpr int PFX_THREADS = 512;
constexpr int PFX_ITEMS = 4;
constexpr int PFX_TILE = PFX_THREADS * PFX_ITEMS;     // 2048 bins per prefix tile

size_t snr_hdr_bytes();

// ------------------------------------------------------------------------- 128-bit fixed point
struct U128 { uint64_t lo, hi; };

__device__ __forceinline__ U128 u128_add(U128 a, U128 b)
{
    U128 r;
    r.lo = a.lo + b.lo;
    r.hi = a.hi + b.hi + (r.lo < a.lo ? 1ull : 0ull);
    return r;
}
__device__ __forceinline__ U128 u128_sub(U128 a, U128 b)
{
    U128 r;
    r.lo = a.lo - b.lo;
    r.hi = a.hi - b.hi - (a.lo < b.lo ? 1ull : 0ull);
    return r;
}
__device__ __forceinline__ U128 u128_shfl_up(U128 v, int o)
{
    U128 r;
    r.lo = __shfl_up_sync(0xffffffffu, v.lo, o);
    r.hi = __shfl_up_sync(0xffffffffu, v.hi, o);
    return r;
}

// Header of the prefix: unit_exp = exponent U of one fixed-point unit (value = integer * 2^U),
// e_top = bound on the terms (every term < 2^e_top), bad = some term was not representable.
struct PrefixHeader { int unit_exp; int e_top; int bad; int pad; };

// x = 1/psd as fixed point with unit 2^U, truncated.  ok = 0 when x is negative, not finite or >= 2^e_top.
__device__ __forceinline__ U128 inv_to_fixed(double psd, int U, int e_top, int *ok)
{
    const double x = __drcp_rn(psd);                        // the correctly rounded 1 / psd, as the division gives
    const long long bits = __double_as_longlong(x);
    const int e = (int)((bits >> 52) & 0x7ff);
    U128 v; v.lo = 0; v.hi = 0;
    if (bits < 0 || e == 0x7ff || e - 1022 > e_top) { *ok = 0; return v; }
    if (e == 0) return v;                                   // zero / subnormal: below one unit anyway
    const uint64_t mant = ((uint64_t)bits & 0x000fffffffffffffull) | 0x0010000000000000ull;
    const int sh = (e - 1075) - U;                          // x = mant * 2^(e - 1075)
    if (sh >= 0) {
        if (sh >= 64) { v.hi = mant << (sh - 64); }
        else { v.lo = mant << sh; v.hi = sh ? (mant >> (64 - sh)) : 0ull; }
    } else if (sh > -64) {
        v.lo = mant >> (-sh);
    }
    return v;
}

// integer * 2^U -> binary64, round to nearest
__device__ __forceinline__ double fixed_to_double(U128 d, int U)
{
    if (d.hi == 0) return ldexp(__ull2double_rn(d.lo), U);
    const int lz = __clzll((long long)d.hi);
    uint64_t top = lz ? ((d.hi << lz) | (d.lo >> (64 - lz))) : d.hi;
    const uint64_t rest = lz ? (d.lo << lz) : d.lo;
    if (rest) top |= 1ull;                                  // sticky bit
    return ldexp(__ull2double_rn(top), U + 64 - lz);
}

// e_top from the largest 1/arr[k] of the grid (arr = s_instr in the loop, psd in the stage call).
// Grid-wide: every CTA folds its maximum into the scratch words behind the header (zero on entry);
// the last CTA to finish writes the header and clears the scratch.
struct PrefixScratch { int emax_biased; int bad; unsigned ticket; int pad; };   // emax_biased = e + 200000, 0 = none

__global__ void __launch_bounds__(256)
prefix_header_kernel(const double *__restrict__ arr, int64_t n, int64_t n_bins_row, PrefixHeader *hdr)
{
    __shared__ int wmax[8], wbad[8];
    PrefixScratch *sc = reinterpret_cast<PrefixScratch *>(hdr + 1);
    int emax = -100000;
    int bad = 0;
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    for (int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; k < n; k += stride) {
        const double x = __drcp_rn(arr[k]);
        const long long bits = __double_as_longlong(x);
        const int e = (int)((bits >> 52) & 0x7ff);
        if (bits < 0 || e == 0x7ff) bad = 1;
        else if (e - 1022 > emax) emax = e - 1022;
    }
    for (int o = 16; o; o >>= 1) {
        emax = max(emax, __shfl_xor_sync(0xffffffffu, emax, o));
        bad |= __shfl_xor_sync(0xffffffffu, bad, o);
    }
    if ((threadIdx.x & 31) == 0) { wmax[threadIdx.x >> 5] = emax; wbad[threadIdx.x >> 5] = bad; }
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int w = 1; w < (int)(blockDim.x >> 5); ++w) { emax = max(emax, wmax[w]); bad |= wbad[w]; }
        if (emax > -100000) atomicMax(&sc->emax_biased, emax + 200000);
        if (bad) atomicOr(&sc->bad, 1);
        __threadfence();
        if (atomicAdd(&sc->ticket, 1u) == gridDim.x - 1) {
            __threadfence();
            const int eb = atomicAdd(&sc->emax_biased, 0);
            const int anybad = atomicAdd(&sc->bad, 0);
            int L = 0;
            while (((int64_t)1 << L) < n_bins_row) ++L;
            PrefixHeader h;
            h.bad = (anybad || eb == 0) ? 1 : 0;
            h.e_top = h.bad ? 0 : eb - 200000;
            h.unit_exp = h.e_top + L - 127;
            h.pad = 0;
            *hdr = h;
            sc->emax_biased = 0; sc->bad = 0; sc->ticket = 0u;
        }
    }
}

// Local inclusive prefix of every tile of PFX_TILE bins + the tile totals (no prefix across tiles: a sum over a
// stretch of bins is a difference of two local prefixes plus the totals of the tiles it crosses, rho2_of); skipped for
// tiles without a dirty block: their prefix stands).  gridDim.x CTAs per row, resident together; CTA b
// takes the tiles b, b + gridDim.x, ...: 32 of them are looked up at once (lane l the l-th), so a pass
// with a handful of dirty tiles costs one look-up per CTA, not one CTA per tile.
__global__ void __launch_bounds__(PFX_THREADS, 3)
inv_prefix_local_kernel(const double *__restrict__ psd, int64_t n_bins, int tiles_per_row,
                        U128 *__restrict__ pref, U128 *__restrict__ tile_tot, PrefixHeader *hdr, DirtyView dv)
{
    __shared__ U128 wtot[PFX_THREADS / 32];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    gbfg_let_next_kernel_start();
    gbfg_wait_prior_kernel();                               // the PSD of this pass
    const int *cum = dv.cum ? dv.cum + (int64_t)blockIdx.y * (dv.n_dblk + 1) : nullptr;
    const int64_t row = (int64_t)blockIdx.y * n_bins;
    int ok = 1;
    const int U = hdr->unit_exp, e_top = hdr->e_top;        // in flight together with the first dirty look-up
    static_assert(PFX_ITEMS == 4, "one 256-bit vector of psd per thread");
    const bool vec_row = ((((uintptr_t)(psd + row)) | ((uintptr_t)(pref + row))) & 31u) == 0;
    for (int t0 = blockIdx.x; t0 < tiles_per_row; t0 += 32 * gridDim.x) {
        const int t_mine = t0 + lane * gridDim.x;
        bool dirty = t_mine < tiles_per_row;
        if (dirty && cum) {                                 // psd of this tile unchanged: its prefix stands
            const int64_t k_first = (int64_t)t_mine * PFX_TILE;
            int64_t k_last = k_first + PFX_TILE - 1;
            if (k_last > n_bins - 1) k_last = n_bins - 1;
            dirty = cum[(k_last >> dv.dblk_log2) + 1] != cum[k_first >> dv.dblk_log2];
        }
        for (unsigned todo = __ballot_sync(0xffffffffu, dirty); todo; todo &= todo - 1) {
            const int tile = t0 + (__ffs(todo) - 1) * gridDim.x;
            const int64_t base = (int64_t)tile * PFX_TILE + (int64_t)threadIdx.x * PFX_ITEMS;
            // a thread's four bins are one 32-byte sector of psd and two of the prefix: moved as 256-bit vectors where
            // the row allows it (with narrower accesses every sector is touched four times and the L1 is what limits)
            const bool vec = vec_row && base + PFX_ITEMS <= n_bins;
            double x[PFX_ITEMS];
            if (vec) {
                asm volatile("ld.global.v4.f64 {%0, %1, %2, %3}, [%4];" : "=d"(x[0]), "=d"(x[1]), "=d"(x[2]), "=d"(x[3]) : "l"(psd + row + base) : "memory");
            } else {
#pragma unroll
                for (int j = 0; j < PFX_ITEMS; ++j) x[j] = base + j < n_bins ? psd[row + base + j] : 0.0;
            }
            U128 v[PFX_ITEMS];
            U128 run; run.lo = 0; run.hi = 0;
#pragma unroll
            for (int j = 0; j < PFX_ITEMS; ++j) {
                const int64_t k = base + j;
                U128 t; t.lo = 0; t.hi = 0;
                if (k < n_bins) t = inv_to_fixed(x[j], U, e_top, &ok);
                run = u128_add(run, t);
                v[j] = run;
            }
            U128 incl = run;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                U128 up = u128_shfl_up(incl, o);
                if (lane >= o) incl = u128_add(incl, up);
            }
            __syncthreads();                                // the last tile's readers of wtot are done
            if (lane == 31) wtot[warp] = incl;
            __syncthreads();
            U128 before = u128_sub(incl, run);
            for (int w = 0; w < warp; ++w) before = u128_add(before, wtot[w]);
            if (vec) {
#pragma unroll
                for (int j = 0; j < PFX_ITEMS; j += 2) {
                    const U128 a0 = u128_add(before, v[j]), a1 = u128_add(before, v[j + 1]);
                    asm volatile("st.global.v4.u64 [%0], {%1, %2, %3, %4};" ::"l"(pref + row + base + j), "l"(a0.lo), "l"(a0.hi), "l"(a1.lo), "l"(a1.hi) : "memory");
                }
            } else {
#pragma unroll
                for (int j = 0; j < PFX_ITEMS; ++j) {
                    const int64_t k = base + j;
                    if (k < n_bins) pref[row + k] = u128_add(before, v[j]);
                }
            }
            if (threadIdx.x == PFX_THREADS - 1) tile_tot[(int64_t)blockIdx.y * tiles_per_row + tile] = u128_add(before, run);
        }
    }
    if (!ok) hdr->bad = 1;
}

// sum of the fixed-point terms of the bins [k0, k0 + w) of a row: local prefixes at both ends + the totals of the tiles
// in between (integers: the same bits in whatever order they are added)
__device__ __forceinline__ U128 prefix_range(const U128 *__restrict__ pref, const U128 *__restrict__ tile_tot,
                                             int64_t row_bin0, int64_t row_tile0, int64_t k0, int64_t w)
{
    const int64_t k1 = k0 + w - 1;
    U128 sum = pref[row_bin0 + k1];
    int64_t t = 0;
    if (k0 > 0) {
        sum = u128_sub(sum, pref[row_bin0 + k0 - 1]);
        t = (k0 - 1) / PFX_TILE;
    }
    for (const int64_t t1 = k1 / PFX_TILE; t < t1; ++t) sum = u128_add(sum, tile_tot[row_tile0 + t]);
    return sum;
}

// What the test needs of the prefix (all NULL / 0: direct sums only)
struct PrefixView {
    const U128 *pref;           // [rows][n_bins] local inclusive prefixes
    const U128 *tile_tot;       // [rows][tiles_per_row] tile totals
    const PrefixHeader *hdr;
    int tiles_per_row;
};

// sum over [gk0, gk0 + w) of four_p / psd (psd, pref indexed by global bin; row = its catalog row)
__device__ __forceinline__ double rho2_direct(const double *__restrict__ psd, int64_t gk0, int64_t w, double four_p)
{
    double acc = 0.0;
    for (int64_t k = gk0; k < gk0 + w; ++k) acc = acc + four_p / psd[k];
    return acc;
}

__device__ __forceinline__ double rho2_of(const double *__restrict__ psd, const PrefixView &pv, bool pref_ok, int unit_exp,
                                          int64_t gk0, int64_t w, int64_t n_bins, int row, double four_p, bool *exact)
{
    *exact = true;
    if (w <= SNR_NARROW || !pref_ok) return rho2_direct(psd, gk0, w, four_p);
    const int64_t row_bin0 = (int64_t)row * n_bins, row_tile0 = (int64_t)row * pv.tiles_per_row;
    const int64_t k0 = gk0 - row_bin0;
    const U128 hi = prefix_range(pv.pref, pv.tile_tot, row_bin0, row_tile0, k0, w);
    // every term was truncated by less than one unit: keep the relative error under 2^-46
    if (hi.hi == 0 && hi.lo < ((uint64_t)w << 46)) return rho2_direct(psd, gk0, w, four_p);
    *exact = false;
    return four_p * fixed_to_double(hi, unit_exp);
}

// source index (< 2^36) and place inside the bucket (< 2^28) of a record as first compacted
constexpr int CAND_SLOT_SHIFT = 36;
constexpr int64_t CAND_SRC_MASK = ((int64_t)1 << CAND_SLOT_SHIFT) - 1;

struct CandArrays {
    int64_t *gk0;       // first bin, as index into the [n_cat][n_bins] arrays
    int32_t *w;         // w_eff; set to 0 once the source is resolved
    double *four_p;
    int64_t *src;       // global source index
};

struct BuildArgs {
    const double *A, *f, *fdot;
    const uint8_t *resolved;
    const double *s_instr;      // [n_bins], NULL: keep every valid unresolved source (no pre-selection)
    PrefixView pv;              // prefix of 1/s_instr (one row)
    double thr_pre;             // rho_th^2 (1 - 4e-9)
    double *rho2_out;           // nullable: NaN is written for rejected sources
    CandArrays cand;
    int64_t *cand_count;        // [1 + n_cat]: total, per catalog
    int64_t i_begin, n_all;     // sources [i_begin, n_all) of the batch
    int *bkt_count, *bkt_ext;   // [n_cat][n_dblk]: zero on entry
    int n_dblk, dblk_log2;
};

// CTA_APPEND: one append to the candidate counter per CTA and trip instead of one per warp (batches of 1e8 sources)
template <bool CTA_APPEND>
__global__ void __launch_bounds__(256)
cand_build_kernel(GridDev g, CatTable ct, BuildArgs a)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    const int64_t n_round = a.i_begin + ((a.n_all - a.i_begin + 255) & ~(int64_t)255);   // the same number of trips for every thread of a CTA
    // CTA_APPEND: a batch of 3e8 sources would otherwise put 1e7 atomics on one counter
    __shared__ int s_wcnt[2][8];
    __shared__ long long s_base[2];
    int trip = 0;
    bool pref_ok = false;
    int unit_exp = 0;
    if (a.s_instr && a.pv.pref) { pref_ok = a.pv.hdr->bad == 0; unit_exp = a.pv.hdr->unit_exp; }
    for (int64_t i = a.i_begin + (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n_round; i += stride) {
        bool keep = false;
        SrcBins s; s.status = 1; s.k0 = 0; s.w_eff = 0; s.p = 0.0; s.q = 0;
        int cat = 0;
        if (i < a.n_all && a.resolved[i] == 0) {
            s = source_bins(g, a.A[i], a.f[i], a.fdot[i]);
            if (s.status == 0) {
                keep = true;
                if (ct.n_cat > 1) cat = cat_of(ct, i);
                if (a.s_instr) {
                    bool exact;
                    const double r2 = rho2_of(a.s_instr, a.pv, pref_ok, unit_exp, s.k0, s.w_eff, g.n_bins, 0, 4.0 * s.p, &exact);
                    keep = r2 > a.thr_pre;
                }
            } else if (a.rho2_out) {
                a.rho2_out[i] = __longlong_as_double(0x7ff8000000000000ll);
            }
        }
        const unsigned mask = __ballot_sync(0xffffffffu, keep);
        const int buf = trip & 1;
        ++trip;
        if (CTA_APPEND) {
            if (lane == 0) s_wcnt[buf][warp] = __popc(mask);
            __syncthreads();
            if (threadIdx.x == 0) {
                int tot = 0;
                for (int w = 0; w < 8; ++w) tot += s_wcnt[buf][w];
                s_base[buf] = tot ? (long long)atomicAdd((unsigned long long *)a.cand_count, (unsigned long long)tot) : 0ll;
            }
            __syncthreads();
        }
        if (mask) {
            int64_t base = 0;
            if (CTA_APPEND) {
                base = s_base[buf];
                for (int w = 0; w < warp; ++w) base += s_wcnt[buf][w];
            } else {
                if (lane == 0) base = (int64_t)atomicAdd((unsigned long long *)a.cand_count, (unsigned long long)__popc(mask));
                base = __shfl_sync(0xffffffffu, base, 0);
            }
            const unsigned same = ct.n_cat > 1 ? __match_any_sync(0xffffffffu, keep ? cat : -1) : 0u;   // kept lanes of my catalog
            if (keep) {
                const int64_t t = base + __popc(mask & ((1u << lane) - 1u));
                a.cand.gk0[t] = (int64_t)cat * g.n_bins + s.k0;
                a.cand.w[t] = (int32_t)s.w_eff;
                a.cand.four_p[t] = 4.0 * s.p;
                if (ct.n_cat > 1 && lane == __ffs(same) - 1)   // one add per warp and catalog (a warp rarely straddles two)
                    atomicAdd((unsigned long long *)(a.cand_count + 1 + cat), (unsigned long long)__popc(same));
                const int64_t gb = (int64_t)cat * a.n_dblk + (s.k0 >> a.dblk_log2);
                // the record's place inside its bucket is taken here, so that the ordering pass (cand_scatter_kernel)
                // needs no atomics of its own: it rides in the upper bits of the source index
                const int64_t slot = atomicAdd(a.bkt_count + gb, 1);
                a.cand.src[t] = i | (slot << CAND_SLOT_SHIFT);
                atomicMax(a.bkt_ext + gb, (int)((s.k0 + s.w_eff - 1) >> a.dblk_log2));
            }
        }
    }
}

// Buckets = (row, dirty block of the first bin).  One CTA per row: first record of every bucket
// (exclusive scan of the counts, on top of the records of the rows before), the scatter cursors,
// and the prefix maximum of the last block reached.
constexpr int BKT_THREADS = 1024;

__global__ void __launch_bounds__(BKT_THREADS)
cand_bucket_scan_kernel(int *__restrict__ bkt_count, int *__restrict__ bkt_ext, int64_t *__restrict__ bkt_off,
                        const int64_t *__restrict__ cand_count, int n_dblk)
{
    __shared__ int wsum[32], wmax[32];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int row = blockIdx.x;
    int64_t base = 0;
    if (gridDim.x > 1) for (int c = 0; c < row; ++c) base += cand_count[1 + c];
    int *cnt = bkt_count + (int64_t)row * n_dblk;
    int *ext = bkt_ext + (int64_t)row * n_dblk;
    int64_t *off = bkt_off + (int64_t)row * (n_dblk + 1);
    // a thread's buckets (at most 16: n_dblk <= DIRTY_MAX_BLOCKS) are read once, all loads in flight together; the two
    // loops over them used to be chains of 15 dependent round trips each
    constexpr int PER_MAX = DIRTY_MAX_BLOCKS / BKT_THREADS;
    const int per = (n_dblk + BKT_THREADS - 1) / BKT_THREADS;
    const int b_lo = min(tid * per, n_dblk), b_hi = min(b_lo + per, n_dblk);
    int c_[PER_MAX], e_[PER_MAX];
#pragma unroll
    for (int u = 0; u < PER_MAX; ++u) {
        const int b = b_lo + u;
        c_[u] = b < b_hi ? cnt[b] : 0;
        e_[u] = b < b_hi ? ext[b] : -1;
    }
    int s = 0, m = -1;
#pragma unroll
    for (int u = 0; u < PER_MAX; ++u) { s += c_[u]; if (c_[u]) m = max(m, e_[u]); }
    int incl = s, imax = m;
    for (int o = 1; o < 32; o <<= 1) {
        const int us = __shfl_up_sync(0xffffffffu, incl, o), um = __shfl_up_sync(0xffffffffu, imax, o);
        if (lane >= o) { incl += us; imax = max(imax, um); }
    }
    if (lane == 31) { wsum[warp] = incl; wmax[warp] = imax; }
    __syncthreads();
    int run = incl - s;
    int pm = __shfl_up_sync(0xffffffffu, imax, 1);
    if (lane == 0) pm = -1;
    for (int w = 0; w < warp; ++w) { run += wsum[w]; pm = max(pm, wmax[w]); }
#pragma unroll
    for (int u = 0; u < PER_MAX; ++u) {
        const int b = b_lo + u;
        if (b < b_hi) {
            off[b] = base + run;
            cnt[b] = 0;                                // becomes the scatter cursor (relative to off[b])
            if (c_[u]) pm = max(pm, e_[u]);
            ext[b] = pm;
            run += c_[u];
        }
    }
    if (tid == BKT_THREADS - 1) off[n_dblk] = base + run;
}

// reach[b] = first bucket whose records reach block b = first index with prefix maximum >= b (n_dblk: none)
__global__ void __launch_bounds__(256)
cand_bucket_reach_kernel(const int *__restrict__ bkt_pm, int *__restrict__ bkt_reach, int n_dblk)
{
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= n_dblk) return;
    const int *pm = bkt_pm + (int64_t)blockIdx.y * n_dblk;
    int lo = 0, hi = n_dblk;
    while (lo < hi) { const int mid = (lo + hi) >> 1; if (pm[mid] >= b) hi = mid; else lo = mid + 1; }
    bkt_reach[(int64_t)blockIdx.y * n_dblk + b] = lo;
}

struct CandArraysConst { const int64_t *gk0; const int32_t *w; const double *four_p; const int64_t *src; };

__device__ __forceinline__ void store_rec(CandRec *p, int64_t gk0, double four_p, int64_t src, int32_t w)
{
    asm volatile("st.global.v4.u64 [%0], {%1, %2, %3, %4};" ::"l"(p), "l"(gk0), "l"(__double_as_longlong(four_p)), "l"(src),
                 "l"((int64_t)(uint32_t)w) : "memory");
}
__device__ __forceinline__ void load_rec(const CandRec *p, int64_t &gk0, double &four_p, int64_t &src, int32_t &w)
{
    int64_t fp, wp;
    asm volatile("ld.global.v4.u64 {%0, %1, %2, %3}, [%4];" : "=l"(gk0), "=l"(fp), "=l"(src), "=l"(wp) : "l"(p) : "memory");
    four_p = __longlong_as_double(fp);
    w = (int32_t)(uint32_t)wp;
}

__global__ void __launch_bounds__(256)
cand_scatter_kernel(CandArraysConst in, CandRec *__restrict__ out, const int64_t *__restrict__ cand_count, int *__restrict__ bkt_cur,
                    const int64_t *__restrict__ bkt_off, int64_t n_bins, int n_dblk, int dblk_log2)
{
    const int64_t n = *cand_count;
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    for (int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; t < n; t += stride) {
        const int64_t gk0 = in.gk0[t];
        const int64_t row = gk0 / n_bins;
        const int64_t b = (gk0 - row * n_bins) >> dblk_log2;
        const int64_t packed = in.src[t];
        const int64_t dst = bkt_off[row * (n_dblk + 1) + b] + (packed >> CAND_SLOT_SHIFT);
        store_rec(out + dst, gk0, in.four_p[t], packed & CAND_SRC_MASK, in.w[t]);
    }
}

struct SnrArgs {
    const double *psd;          // [n_cat][n_bins]
    PrefixView pv;              // prefix of 1/psd
    CandRec *rec;              // the ordered records
    const int64_t *cand_count;
    const int *abort_flag;      // nullable: when *abort_flag != 0 the kernel does nothing (loop.cu)
    DirtyView dv;               // cum != NULL: a candidate whose bins lie in clean blocks is not re-tested
    const int64_t *bkt_off;     // [n_cat][n_dblk + 1] first record of each bucket
    const int *bkt_reach;       // [n_cat][n_dblk] first bucket with a record that reaches block b
    int *any_near;
    int n_dblk;
    int64_t *test_count;        // [n_cat] tests evaluated, accumulated (nullable)
    SubtractView sub;           // spectrum != NULL: a selected source is subtracted on the spot (eq. D4)
    const unsigned long long *delta_bits;   // nullable: [n_cat] PSD change of this pass; a row at or under psd_rtol is frozen (R13)
    double psd_rtol;
    int64_t n_bins;
    int n_cat;
    double thr;                 // rho_th^2
    uint8_t *resolved;
    double *rho2_out;           // nullable
    int64_t *sel_idx;
    int64_t *sel_count;         // [1 + n_cat]
    int64_t *near_count;        // nullable; one counter, or one per catalog
    int near_per_cat;
};

__global__ void __launch_bounds__(256)
snr_cand_kernel(SnrArgs a)
{
    gbfg_wait_prior_kernel();                               // the prefix of this pass
    // every look-up that does not depend on another one is issued before the first is used (a late pass is a
    // chain of L2 round trips, not work)
    const int rowc = blockIdx.y;
    const int64_t *off = a.bkt_off + (int64_t)rowc * (a.n_dblk + 1);
    const int abort_v = a.abort_flag ? *a.abort_flag : 0;
    const unsigned long long dbits = a.delta_bits ? a.delta_bits[rowc] : 0ull;
    const int near_v = a.dv.cum ? a.any_near[0] : 1;     // launch-invariant: raised flags go to word 1
    const int b_min = a.dv.cum ? a.dv.range[2 * rowc] : 0, b_max = a.dv.cum ? a.dv.range[2 * rowc + 1] : 0;
    const int hdr_bad = a.pv.pref ? a.pv.hdr->bad : 1;
    const int unit_exp = a.pv.pref ? a.pv.hdr->unit_exp : 0;
    int64_t t_first = off[0], n = off[a.n_dblk];
    if (abort_v) return;
    if (a.delta_bits && __longlong_as_double((long long)dbits) <= a.psd_rtol) return;   // S_n has converged
    const int lane = threadIdx.x & 31;
    // records of row blockIdx.y, narrowed to the buckets that can reach a dirty block
    if (a.dv.cum && near_v == 0) {
        if (b_min > b_max) return;                          // nothing dirty in this row
        const int64_t n_hi = off[b_max + 1];
        const int first_bucket = a.bkt_reach[(int64_t)rowc * a.n_dblk + b_min];
        if (first_bucket >= a.n_dblk) return;
        t_first = off[first_bucket];
        n = n_hi;
    }
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    const bool pref_ok = hdr_bad == 0;
    // The selected indices of the CTA are collected in shared memory and appended to the list with
    // one global atomic per flush (tens of thousands of sources pass in the first iterations: one
    // atomic per warp on a single address is what the kernel then waits for).
    __shared__ int64_t s_sel[SNR_SEL_CAP];
    __shared__ int s_n, s_near, s_tests;
    __shared__ long long s_base;
    if (threadIdx.x == 0) { s_n = 0; s_near = 0; s_tests = 0; }
    __syncthreads();
    for (int64_t t0 = t_first + (int64_t)blockIdx.x * blockDim.x; t0 < n; t0 += stride) {
        const int64_t t = t0 + threadIdx.x;
        int32_t w = 0;
        int64_t src = -1, gk0 = 0, rec_src = -1;
        double four_p = 0.0;
        if (t < n) load_rec(a.rec + t, gk0, four_p, rec_src, w);
        bool sel = false, near = false;
        const int cat = rowc;
        const bool always = w < 0;                          // was near the threshold: counted every iteration
        if (always) w = -w;
        if (w > 0) {
            if (a.dv.cum && !always) {
                // the PSD under this source is what it was at its last test: same rho2, same answer
                const int64_t k0 = gk0 - (int64_t)cat * a.n_bins;
                const int *cum = a.dv.cum + (int64_t)cat * (a.dv.n_dblk + 1);
                if (cum[((k0 + w - 1) >> a.dv.dblk_log2) + 1] == cum[k0 >> a.dv.dblk_log2]) w = 0;
            }
        }
        if (w > 0) {
            bool exact;
            double r2 = rho2_of(a.psd, a.pv, pref_ok, unit_exp, gk0, w, a.n_bins, cat, four_p, &exact);
            if (!exact && fabs(r2 / a.thr - 1.0) <= 4e-9) r2 = rho2_direct(a.psd, gk0, w, four_p);   // decide on the definition's sum
            near = fabs(r2 / a.thr - 1.0) <= 2e-9;
            sel = r2 > a.thr;
            if (a.rho2_out || sel) src = rec_src;
            if (a.rho2_out) a.rho2_out[src] = r2;
        }
        const unsigned sel_mask = __ballot_sync(0xffffffffu, sel);
        const unsigned near_mask = __ballot_sync(0xffffffffu, near);
        if (a.test_count) {
            const unsigned test_mask = __ballot_sync(0xffffffffu, w > 0);
            if (test_mask && lane == 0) atomicAdd(&s_tests, __popc(test_mask));
        }
        if (sel_mask) {
            // a place in the CTA's buffer; once that is full (rare: > SNR_SEL_CAP selected by one CTA) straight into the list
            int base = 0;
            if (lane == 0) base = atomicAdd(&s_n, __popc(sel_mask));
            base = __shfl_sync(0xffffffffu, base, 0);
            const int mine = base + __popc(sel_mask & ((1u << lane) - 1u));
            long long gbase = 0;
            const int n_over = base + __popc(sel_mask) - SNR_SEL_CAP;     // > 0: that many of this warp's do not fit
            if (n_over > 0 && lane == 0) {
                const int cnt = n_over < __popc(sel_mask) ? n_over : __popc(sel_mask);
                gbase = (long long)atomicAdd((unsigned long long *)a.sel_count, (unsigned long long)cnt);
                atomicAdd((unsigned long long *)(a.sel_count + 1 + rowc), (unsigned long long)cnt);
            }
            gbase = __shfl_sync(0xffffffffu, gbase, 0);
            if (sel) {
                if (mine < SNR_SEL_CAP) s_sel[mine] = src;
                else a.sel_idx[gbase + (mine - (base > SNR_SEL_CAP ? base : SNR_SEL_CAP))] = src;
                a.resolved[src] = 1;
                a.rec[t].w = 0;
            }
        }
        if (sel && a.sub.spectrum) {
            // stage (v), eq. (D4): spectrum[k] -= q over the source's bins, in the range-update form of deposit.cu
            // (q from p = four_p / 4, exactly the deposit's), and the blocks whose median can change are stamped
            const int64_t q = __double2ll_rn(ldexp(0.25 * four_p, -a.sub.scale_log2));
            if (q != 0) {
                const int64_t k0 = gk0 - (int64_t)cat * a.n_bins;
                const DepositMarks &mk = a.sub.mk;
                if (w <= DEP_NARROW) {
                    for (int k = 0; k < w; ++k) atomic_add_i64(a.sub.spectrum + gk0 + k, -q);
                } else {
                    const int64_t t_lo = (int64_t)cat * mk.scan_tiles + k0 / DEP_SCAN_TILE;
                    atomic_add_i64(a.sub.diff + gk0, -q);
                    mk.scan_stamp[t_lo] = mk.stamp;
                    if (mk.live_sums) atomic_add_i64(mk.live_sums + t_lo, -q);
                    if (k0 + w < a.n_bins) {
                        const int64_t t_hi = (int64_t)cat * mk.scan_tiles + (k0 + w) / DEP_SCAN_TILE;
                        atomic_add_i64(a.sub.diff + gk0 + w, q);
                        mk.scan_stamp[t_hi] = mk.stamp;
                        if (mk.live_sums) atomic_add_i64(mk.live_sums + t_hi, q);
                    }
                    *a.sub.wide_flag = mk.stamp;
                }
                if (mk.blk_stamp) {
                    int64_t lo = k0 - mk.med_h, hi = k0 + w - 1 + mk.med_h;
                    if (lo < 0) lo = 0;
                    if (hi > a.n_bins - 1) hi = a.n_bins - 1;
                    int *bs = mk.blk_stamp + (int64_t)cat * mk.n_dblk;
                    for (int64_t b = lo >> mk.dblk_log2; b <= (hi >> mk.dblk_log2); ++b) bs[b] = mk.stamp;
                }
            }
        }
        if (near && !sel && !always) { a.rec[t].w = -w; a.any_near[1] = 1; }
        if (near_mask && lane == 0) atomicAdd(&s_near, __popc(near_mask));
    }
    // one append per CTA for what its buffer holds
    __syncthreads();
    {
        const int cnt = s_n < SNR_SEL_CAP ? s_n : SNR_SEL_CAP;
        if (cnt > 0) {
            if (threadIdx.x == 0) {
                s_base = (long long)atomicAdd((unsigned long long *)a.sel_count, (unsigned long long)cnt);
                atomicAdd((unsigned long long *)(a.sel_count + 1 + rowc), (unsigned long long)cnt);
            }
            __syncthreads();
            for (int i = threadIdx.x; i < cnt; i += blockDim.x) a.sel_idx[s_base + i] = s_sel[i];
        }
    }
    if (threadIdx.x == 0 && a.test_count && s_tests) atomicAdd((unsigned long long *)(a.test_count + rowc), (unsigned long long)s_tests);
    if (threadIdx.x == 0 && s_near && a.near_count)
        atomicAdd((unsigned long long *)(a.near_count + (a.near_per_cat ? rowc : 0)), (unsigned long long)s_near);
}

// ---------------------------------------------------------------------------------------------
// internal entries (used by the stage call and by the loop, loop.cu)
// ---------------------------------------------------------------------------------------------
int pfx_tiles_per_row(int64_t n_bins) { return (int)((n_bins + PFX_TILE - 1) / PFX_TILE); }

static PrefixView make_view(const SnrWork &sw, int64_t n_bins)
{
    PrefixView pv;
    pv.pref = (const U128 *)sw.pref;
    pv.tile_tot = (const U128 *)sw.tile_tot;
    pv.hdr = (const PrefixHeader *)sw.hdr;
    pv.tiles_per_row = pfx_tiles_per_row(n_bins);
    return pv;
}

// hdr <- scale of the fixed-point prefix, from the largest 1/arr[k]; arr: [n], rows of n_bins_row
int launch_prefix_header(const double *arr, int64_t n, int64_t n_bins_row, const SnrWork &sw, cudaStream_t st)
{
    GBFG_CUDA(cudaMemsetAsync(sw.hdr, 0, snr_hdr_bytes(), st));
    int64_t blocks = (n + 255) / 256;
    const int64_t cap = (int64_t)sm_count() * 8;
    if (blocks > cap) blocks = cap;
    if (blocks < 1) blocks = 1;
    LaunchTimer lt(K_INV_BLOCKS, st);
    prefix_header_kernel<<<(int)blocks, 256, 0, st>>>(arr, n, n_bins_row, (PrefixHeader *)sw.hdr);
    GBFG_LAUNCH_CHECK("prefix_header_kernel");
    return GBFG_OK;
}

// prefix of 1/psd for every row; dv.cum != NULL: only the tiles that hold a dirty block are redone
// (the others must hold the prefix of an earlier call on the same psd values)
int launch_inv_prefix(const double *psd, int64_t n_bins, int n_cat, const SnrWork &sw, const DirtyView &dv, cudaStream_t st)
{
    const int tiles = pfx_tiles_per_row(n_bins);
    int per_row = (3 * sm_count() + n_cat - 1) / n_cat;        // three CTAs per SM over all rows;
    if (per_row < 64) per_row = 64;                            // a batch: more, shorter CTAs (rows differ in how dirty they are)
    if (per_row > tiles) per_row = tiles;
    LaunchTimer lt(K_INV_BLOCKS, st);
    cudaError_t e = launch_dependent(inv_prefix_local_kernel, dim3(per_row, n_cat), dim3(PFX_THREADS), 0, st, psd, n_bins, tiles,
                                     (U128 *)sw.pref, (U128 *)sw.tile_tot, (PrefixHeader *)sw.hdr, dv);
    if (e != cudaSuccess) return set_cuda_error(e, "inv_prefix_local_kernel");
    GBFG_LAUNCH_CHECK("inv_prefix_local_kernel");
    return GBFG_OK;
}

// candidate records of every unresolved valid source; s_instr != NULL: pre-selection against the
// instrument noise (the prefix in sw must then be that of 1/s_instr, one row).
// sw.cand_count[0 .. n_cat] must be zero on entry.
// Three steps, so that the records of a catalog can be built piece by piece while it is still being drawn (loop.cu):
// begin (clears the bucket counts), any number of ranges [i_begin, i_end) of the batch, finish (orders the records).
int cand_build_begin(const CatTable &ct, int64_t n_bins, const SnrWork &sw, cudaStream_t st)
{
    const int n_dblk = dirty_blocks_per_row(n_bins);
    GBFG_CUDA(cudaMemsetAsync(sw.bkt_count, 0, sizeof(int) * (size_t)ct.n_cat * (size_t)n_dblk, st));
    GBFG_CUDA(cudaMemsetAsync(sw.bkt_ext, 0, sizeof(int) * (size_t)ct.n_cat * (size_t)n_dblk, st));
    GBFG_CUDA(cudaMemsetAsync(sw.any_near, 0, 2 * sizeof(int), st));
    return GBFG_OK;
}

int cand_build_range(const GridDev &g, const CatTable &ct, const double *A, const double *f, const double *fdot,
                     const uint8_t *resolved, const double *s_instr, double rho_th, double *rho2_out,
                     const SnrWork &sw, int64_t i_begin, int64_t i_end, cudaStream_t st)
{
    if (i_end <= i_begin) return GBFG_OK;
    BuildArgs a;
    a.A = A; a.f = f; a.fdot = fdot; a.resolved = resolved; a.s_instr = s_instr;
    a.pv = make_view(sw, g.n_bins);
    a.thr_pre = (rho_th * rho_th) * (1.0 - 4e-9);    // keeps every source the near-threshold count (2e-9) can see
    a.rho2_out = rho2_out;
    a.cand.gk0 = sw.tmp_gk0; a.cand.w = sw.tmp_w; a.cand.four_p = sw.tmp_4p; a.cand.src = sw.tmp_src;
    a.cand_count = sw.cand_count;
    a.i_begin = i_begin; a.n_all = i_end;
    a.bkt_count = sw.bkt_count; a.bkt_ext = sw.bkt_ext;
    a.n_dblk = dirty_blocks_per_row(g.n_bins); a.dblk_log2 = dirty_block_log2(g.n_bins);
    int64_t blocks = (i_end - i_begin + 255) / 256;
    const int64_t cap = (int64_t)sm_count() * 16;
    if (blocks > cap) blocks = cap;
    LaunchTimer lt(K_SNR, st);
    if (ct.n_cat > 1 || ct.offsets[ct.n_cat] >= 30000000) cand_build_kernel<true><<<(int)blocks, 256, 0, st>>>(g, ct, a);
    else cand_build_kernel<false><<<(int)blocks, 256, 0, st>>>(g, ct, a);
    GBFG_LAUNCH_CHECK("cand_build_kernel");
    return GBFG_OK;
}

int cand_build_finish(const GridDev &g, const CatTable &ct, const SnrWork &sw, cudaStream_t st)
{
    const int64_t n = ct.offsets[ct.n_cat];
    const int n_dblk = dirty_blocks_per_row(g.n_bins), dblk_log2 = dirty_block_log2(g.n_bins);
    int64_t blocks = (n + 255) / 256;
    const int64_t cap = (int64_t)sm_count() * 16;
    if (blocks > cap) blocks = cap;
    if (blocks < 1) blocks = 1;
    LaunchTimer lt(K_SNR, st);
    // order the records by (row, dirty block of the first bin)
    cand_bucket_scan_kernel<<<ct.n_cat, BKT_THREADS, 0, st>>>(sw.bkt_count, sw.bkt_ext, sw.bkt_off, sw.cand_count, n_dblk);
    GBFG_LAUNCH_CHECK("cand_bucket_scan_kernel");
    cand_bucket_reach_kernel<<<dim3((n_dblk + 255) / 256, ct.n_cat), 256, 0, st>>>(sw.bkt_ext, sw.bkt_reach, n_dblk);
    GBFG_LAUNCH_CHECK("cand_bucket_reach_kernel");
    CandArraysConst in = {sw.tmp_gk0, sw.tmp_w, sw.tmp_4p, sw.tmp_src};
    cand_scatter_kernel<<<(int)blocks, 256, 0, st>>>(in, sw.cand_rec, sw.cand_count, sw.bkt_count, sw.bkt_off, g.n_bins, n_dblk, dblk_log2);
    GBFG_LAUNCH_CHECK("cand_scatter_kernel");
    return GBFG_OK;
}

int launch_cand_build(const GridDev &g, const CatTable &ct, const double *A, const double *f, const double *fdot,
                      const uint8_t *resolved, const double *s_instr, double rho_th, double *rho2_out,
                      const SnrWork &sw, cudaStream_t st)
{
    const int64_t n = ct.offsets[ct.n_cat];
    if (n <= 0) return GBFG_OK;
    int rc = cand_build_begin(ct, g.n_bins, sw, st);
    if (!rc) rc = cand_build_range(g, ct, A, f, fdot, resolved, s_instr, rho_th, rho2_out, sw, 0, n, st);
    if (!rc) rc = cand_build_finish(g, ct, sw, st);
    return rc;
}

// the test over the candidate records; n_launch = upper bound of the candidate count (grid sizing).
// sel_count[0 .. n_cat] is accumulated into (zero it for a fresh selection).
int launch_snr_cand(int64_t n_bins, int n_cat, const double *psd, double rho_th, uint8_t *resolved, double *rho2_out,
                    int64_t n_launch, int64_t *sel_idx, int64_t *sel_count, int64_t *near_count, int near_per_cat,
                    const int *abort_flag, bool use_prefix, const SnrWork &sw, const DirtyView &dv, int64_t *test_count,
                    const SubtractView *sub, const unsigned long long *delta_bits, double psd_rtol, cudaStream_t st)
{
    if (n_launch <= 0) return GBFG_OK;
    SnrArgs a;
    a.delta_bits = delta_bits; a.psd_rtol = psd_rtol;
    a.test_count = test_count;
    if (sub) a.sub = *sub; else a.sub.spectrum = nullptr;
    a.dv = dv;
    a.psd = psd;
    a.pv = make_view(sw, n_bins);
    if (!use_prefix) { a.pv.pref = nullptr; a.pv.tile_tot = nullptr; }
    a.rec = sw.cand_rec;
    a.cand_count = sw.cand_count;
    a.abort_flag = abort_flag;
    a.n_bins = n_bins; a.n_cat = n_cat;
    a.thr = rho_th * rho_th;
    a.resolved = resolved; a.rho2_out = rho2_out; a.sel_idx = sel_idx; a.sel_count = sel_count;
    a.near_count = near_count; a.near_per_cat = near_per_cat;
    a.bkt_off = sw.bkt_off; a.bkt_reach = sw.bkt_reach; a.any_near = sw.any_near; a.n_dblk = dirty_blocks_per_row(n_bins);
    int64_t blocks = (n_launch / n_cat + 255) / 256 + 1;   // per row; the rows share the records unevenly: grid-stride
    int64_t cap = (int64_t)sm_count() * 16 / n_cat;
    if (cap < 4) cap = 4;
    if (blocks > cap) blocks = cap;
    LaunchTimer lt(K_SNR, st);
    cudaError_t e = launch_dependent(snr_cand_kernel, dim3((unsigned)blocks, (unsigned)n_cat), dim3(256), 0, st, a);
    if (e != cudaSuccess) return set_cuda_error(e, "snr_cand_kernel");
    GBFG_LAUNCH_CHECK("snr_cand_kernel");
    return GBFG_OK;
}

size_t snr_pref_bytes(int64_t n_bins, int n_cat) { return sizeof(U128) * (size_t)n_cat * (size_t)n_bins; }
size_t snr_tile_off_bytes(int64_t n_bins, int n_cat) { return sizeof(U128) * (size_t)n_cat * (size_t)pfx_tiles_per_row(n_bins); }
size_t snr_hdr_bytes() { return sizeof(PrefixHeader) + sizeof(PrefixScratch) + sizeof(unsigned) * GBFG_MAX_CAT; }   // header, scratch, one ticket per row

}  // namespace gbfg
