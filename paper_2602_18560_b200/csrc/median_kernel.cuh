// median_kernel.cuh — the running-median tile kernel (stage iii), included by median.cu.
//
// running_median_tile_kernel<KeyT, THREADS>:
//   <uint32_t, 512>   the fast variant: two CTAs per SM, so that one tile's sort overlaps the other's
//                     walk (every phase of the tile loop is bound by shared-memory latency and barriers,
//                     not by issue slots).  Keys are the low 32 bits of the biased spectrum values, which
//                     order a tile whenever its values agree in their high 32 bits — spectra in units of
//                     2^-140 strain^2 always do.  A tile that does not is appended to the wide list.
//   <uint64_t, 1024>  full 64-bit keys, one CTA per SM: the tiles of the wide list.
// See median.cu for the algorithm (sort once per tile, count table, coarse states, walk).
#pragma once

#include "gbfg_common.cuh"

namespace gbfg {

constexpr int MED_LT = 8192;                  // positions per tile, halos included
constexpr int MED_PB = 32;                    // position block = outputs per coarse chunk
constexpr int MED_FINE = 8;                   // outputs per walking thread
constexpr int MED_STEP_CAP = 20;              // places a thread steps alone before the warp takes over
constexpr int MED_RB = 128;                   // sorted ranks per bucket
constexpr int MED_NPB = MED_LT / MED_PB;      // 256
constexpr int MED_NRB = MED_LT / MED_RB;      // 64
constexpr int MED_TROW = MED_NPB + 2;         // table row stride in u16 (even: rows stay 4-byte aligned)
constexpr int MED_CROW = 256 + 2;             // radix counter row stride in u16 (one row per warp)
constexpr uint64_t SIGN64 = 0x8000000000000000ull;
constexpr int MED_AUX_U16 = MED_NRB * MED_TROW;   // count table (>= 32 rows of radix counters, >= LT output ranks)

template <typename KeyT>
constexpr size_t median_smem_bytes()
{
    return sizeof(KeyT) * MED_LT             // skey
         + sizeof(uint16_t) * MED_LT         // spos
         + sizeof(uint16_t) * MED_LT         // rop
         + sizeof(uint16_t) * MED_AUX_U16    // radix counters, then the count table, then the output ranks
         + sizeof(uint16_t) * MED_NPB        // coarse medians
         + sizeof(uint32_t) * 40;            // scan partials, varying-bit mask
}

struct MedianArgs {
    const int64_t *x;        // [n_cat][n]
    int64_t *med;            // [n_cat][n]
    const double *s_instr;   // [n] or NULL (no PSD)
    double *psd;             // [n_cat][n] or NULL
    const int4 *items;       // work list (row, first output, outputs, -) or NULL: static tiling of every row
    int *ctr;                // [0] number of items, [1] next item
    int4 *wide_items;        // 32-bit variant: tiles whose values differ in the high word are appended here
    int *wide_ctr;           // [0] number of wide items (appended with atomics)
    int n_cat;
    int *neg_flag;           // nullable: set to 1 when a median is negative
    unsigned long long *delta_bits;   // nullable: [n_cat] largest relative PSD change of the row, as binary64 bits (R13)
    int64_t n;
    int h;
    int S;                   // outputs per tile of the static tiling
    int tiles;
    double norm, scale;      // C and 2^scale_log2
};

// n-th (1-based) set bit of a non-zero mask that has at least n bits set
__device__ __forceinline__ int nth_set_bit(unsigned m, int n)
{
    int pos = 0, c;
    c = __popc(m & 0xffffu); if (n > c) { n -= c; m >>= 16; pos += 16; }
    c = __popc(m & 0xffu);   if (n > c) { n -= c; m >>= 8;  pos += 8; }
    c = __popc(m & 0xfu);    if (n > c) { n -= c; m >>= 4;  pos += 4; }
    c = __popc(m & 0x3u);    if (n > c) { n -= c; m >>= 2;  pos += 2; }
    if (n > (int)(m & 1u)) pos += 1;
    return pos;
}

// lanes of the warp whose 8-bit digit equals this lane's (what match.any computes, from 8 ballots)
__device__ __forceinline__ unsigned same_digit_lanes(unsigned d)
{
    unsigned peers = 0xffffffffu;
#pragma unroll
    for (int b = 0; b < 8; ++b) {
        const bool bit = (d >> b) & 1u;
        const unsigned bal = __ballot_sync(0xffffffffu, bit);
        peers &= bit ? bal : ~bal;
    }
    return peers;
}

// DELTA: also record the largest relative PSD change (the second stop rule, R13); a template parameter so
// that the default kernel carries none of it
template <typename KeyT, int THREADS, bool DELTA>
__global__ void __launch_bounds__(THREADS, THREADS <= 512 ? 2 : 1)
running_median_tile_kernel(MedianArgs a)
{
    constexpr int WARPS = THREADS / 32;
    constexpr int ITEMS = MED_LT / THREADS;               // keys per thread in the sort, at most
    constexpr int GROUPS = WARPS / 8;                      // counter scan: thread t owns digit t / GROUPS, 8 warps
    constexpr bool NARROW = sizeof(KeyT) == 4;
    static_assert(THREADS == 256 * GROUPS, "the counter scan maps one thread to one (digit, 8 warps) group");

    extern __shared__ __align__(16) unsigned char smem_raw[];
    KeyT *skey = reinterpret_cast<KeyT *>(smem_raw);
    uint16_t *spos = reinterpret_cast<uint16_t *>(skey + MED_LT);
    uint16_t *rop = spos + MED_LT;
    uint16_t *aux = rop + MED_LT;                          // radix counters, the count table, the output ranks
    uint16_t *cm = aux + MED_AUX_U16;                      // coarse medians
    uint32_t *misc = reinterpret_cast<uint32_t *>(cm + MED_NPB);
    uint16_t *tab = aux;
    uint16_t *orank = aux;                                 // written by the walk, after the table's last use
    uint32_t *aux32 = reinterpret_cast<uint32_t *>(aux);

    const int tid = threadIdx.x;
    const int warp = tid >> 5, lane = tid & 31;
    const unsigned FULL = 0xffffffffu;
    const unsigned lt_mask = (1u << lane) - 1u;
    const int h = a.h, W = 2 * a.h + 1;
    __shared__ int s_item;
    bool neg = false;
    gbfg_let_next_kernel_start();                        // the wide-tile kernel / the prefix may queue up behind this one
    gbfg_wait_prior_kernel();                            // (launched as a dependent: the 32-bit kernel's wide list)

    // work list: the first item of a CTA is its own index, the following ones come from the ticket counter,
    // drawn just before the epilogue so that the atomic's round trip is hidden behind it (earlier would
    // hand the last items to CTAs that are still busy)
    const int n_items = a.items ? a.ctr[0] : 0;
    int next_item = blockIdx.x;
  for (int64_t turn = blockIdx.x;; turn += gridDim.x) {
    int64_t row, o0;
    int n_out, row_i;
    __syncthreads();                                     // the previous tile's epilogue is done with shared memory
    if (a.items) {
        if (tid == 0) s_item = next_item;
        __syncthreads();
        const int item = s_item;
        if (item >= n_items) break;
        const int4 v = a.items[item];
        row_i = v.x;
        o0 = v.y;
        n_out = v.z;
    } else {
        if (turn >= (int64_t)a.tiles * a.n_cat) break;
        const int64_t r = turn / a.tiles, tile = turn - r * a.tiles;
        row_i = (int)r;
        o0 = tile * a.S;
        n_out = (int)((a.n - o0 < a.S) ? (a.n - o0) : a.S);
    }
    row = (int64_t)row_i * a.n;
    const int Lt = n_out + 2 * h;                        // positions really used
    const int rounds = (Lt + THREADS - 1) / THREADS;     // keys per thread in the sort (<= ITEMS)
    const int LTe = rounds * THREADS;                    // positions sorted

    // ---- stage the tile: position p <-> global bin o0 - h + p, reflected at both ends.
    // Unused positions (Lt <= p < LTe) repeat position 0: they are never inside a window.
    if (tid < 2) misc[32 + tid] = 0u;
    __syncthreads();
    uint64_t key_ref;
    {
        int64_t g0 = o0 - h;
        if (g0 < 0) g0 = -g0 - 1;
        if (g0 >= a.n) g0 = 2 * a.n - 1 - g0;
        key_ref = (uint64_t)a.x[row + g0] ^ SIGN64;
        uint64_t vary = 0;
        for (int p0 = tid; p0 < LTe; p0 += 4 * THREADS) {    // four independent loads in flight per thread
            uint64_t key[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const int p = p0 + u * THREADS;
                key[u] = key_ref;
                if (p < Lt) {
                    int64_t g = o0 - h + p;
                    if (g < 0) g = -g - 1;
                    if (g >= a.n) g = 2 * a.n - 1 - g;
                    key[u] = (uint64_t)__ldg(a.x + row + g) ^ SIGN64;
                }
            }
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const int p = p0 + u * THREADS;
                if (p < LTe) {
                    vary |= key[u] ^ key_ref;
                    skey[p] = (KeyT)key[u];
                    spos[p] = (uint16_t)p;
                }
            }
        }
        const unsigned vlo = __reduce_or_sync(FULL, (unsigned)vary);
        const unsigned vhi = __reduce_or_sync(FULL, (unsigned)(vary >> 32));
        if (lane == 0) {
            if (vlo) atomicOr(&misc[32], vlo);
            if (vhi) atomicOr(&misc[33], vhi);
        }
    }
    __syncthreads();
    const uint64_t vary_all = ((uint64_t)misc[33] << 32) | misc[32];
    if (NARROW && (vary_all >> 32) != 0) {               // 32 bits do not order this tile: leave it to the wide kernel
        if (tid == 0) {
            a.wide_items[atomicAdd(&a.wide_ctr[0], 1)] = make_int4(row_i, (int)o0, n_out, 0);
            if (a.items) next_item = (int)gridDim.x + atomicAdd(&a.ctr[1], 1);
        }
        continue;
    }
    const int n_pass = vary_all ? (64 - __clzll((long long)vary_all) + 7) / 8 : 0;

    // ---- LSD radix sort by key, stable, so that equal keys stay in position order.
    // Warp w owns elements [32 rounds w, 32 rounds (w + 1)) of the current order, 32 consecutive ones per round.
    for (int pass = 0; pass < n_pass; ++pass) {
        const int shift = 8 * pass;
        for (int e = tid; e < WARPS * MED_CROW / 2; e += THREADS) aux32[e] = 0u;
        __syncthreads();
        uint16_t *cw = aux + warp * MED_CROW;
        KeyT k[ITEMS];
        uint32_t pk[ITEMS];                              // position << 16 | place among the warp's keys of the same digit
#pragma unroll
        for (int r = 0; r < ITEMS; ++r) {                // the matches are independent: issue them together
            if (r < rounds) {
                const int e = warp * (32 * rounds) + r * 32 + lane;
                k[r] = skey[e];
                pk[r] = __match_any_sync(FULL, (unsigned)(k[r] >> shift) & 255u);
            }
        }
#pragma unroll
        for (int r = 0; r < ITEMS; ++r) {                // counter updates, round after round
            if (r < rounds) {
                const int e = warp * (32 * rounds) + r * 32 + lane;
                const unsigned d = (unsigned)(k[r] >> shift) & 255u;
                const unsigned peers = pk[r];
                const unsigned base = cw[d];
                __syncwarp();
                const unsigned rank = __popc(peers & lt_mask);
                if (rank == 0) cw[d] = (uint16_t)(base + __popc(peers));
                __syncwarp();
                pk[r] = ((unsigned)spos[e] << 16) | (base + rank);
            }
        }
        __syncthreads();
        {   // exclusive scan of the counters in (digit, warp) order: thread t owns digit t / GROUPS, 8 warps
            const int d = tid / GROUPS, wg = (tid % GROUPS) * 8;
            unsigned v[8], s = 0;
#pragma unroll
            for (int i = 0; i < 8; ++i) { v[i] = aux[(wg + i) * MED_CROW + d]; s += v[i]; }
            unsigned incl = s;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                unsigned up = __shfl_up_sync(FULL, incl, o);
                if (lane >= o) incl += up;
            }
            if (lane == 31) misc[warp] = incl;
            __syncthreads();
            unsigned wt = lane < WARPS ? misc[lane] : 0u, wincl = wt;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                unsigned up = __shfl_up_sync(FULL, wincl, o);
                if (lane >= o) wincl += up;
            }
            const unsigned wprev = __shfl_sync(FULL, wincl - wt, warp);
            unsigned run = wprev + incl - s;
#pragma unroll
            for (int i = 0; i < 8; ++i) { aux[(wg + i) * MED_CROW + d] = (uint16_t)run; run += v[i]; }
        }
        __syncthreads();
#pragma unroll
        for (int r = 0; r < ITEMS; ++r) {
            if (r < rounds) {
                const unsigned d = (unsigned)(k[r] >> shift) & 255u;
                const unsigned dst = (unsigned)cw[d] + (pk[r] & 0xffffu);
                skey[dst] = k[r];
                spos[dst] = (uint16_t)(pk[r] >> 16);
            }
        }
        __syncthreads();
    }

    // ---- inverse permutation and the count table (only the rank buckets and position blocks the tile has)
    const int nrb = LTe / MED_RB, npb = LTe / MED_PB;     // LTe is a multiple of 256
    for (int e = tid; e < nrb * MED_TROW / 2; e += THREADS) aux32[e] = 0u;
    __syncthreads();
    for (int r = tid; r < LTe; r += THREADS) {
        int p = spos[r];
        rop[p] = (uint16_t)r;
        int e = (r / MED_RB) * MED_TROW + (p / MED_PB) + 1;
        atomicAdd(&aux32[e >> 1], (e & 1) ? 0x10000u : 1u);
    }
    __syncthreads();
    // prefix along the position blocks: tab[rb][pb] = #{r in bucket rb : pos < pb*PB}
    {
        constexpr int PER = (MED_NPB + 1 + 31) / 32;     // 9 entries per lane
        for (int rb = warp; rb < nrb; rb += WARPS) {
            uint16_t *rowp = tab + rb * MED_TROW;
            int v[PER], s = 0;
#pragma unroll
            for (int q = 0; q < PER; ++q) {
                int idx = lane * PER + q;
                v[q] = idx <= npb ? rowp[idx] : 0;
                s += v[q];
            }
            int incl = s;
            for (int o = 1; o < 32; o <<= 1) {
                int up = __shfl_up_sync(FULL, incl, o);
                if (lane >= o) incl += up;
            }
            int run = incl - s;
#pragma unroll
            for (int q = 0; q < PER; ++q) {
                int idx = lane * PER + q;
                run += v[q];
                if (idx <= npb) rowp[idx] = (uint16_t)run;
            }
        }
    }
    __syncthreads();
    // exclusive prefix along the rank buckets: tab[rb][pb] = #{r < rb*RB : pos < pb*PB}
    for (int pb = tid; pb <= npb; pb += THREADS) {
        int run = 0;
        for (int rb = 0; rb < nrb; ++rb) {
            int v = tab[rb * MED_TROW + pb];
            tab[rb * MED_TROW + pb] = (uint16_t)run;
            run += v;
        }
    }
    __syncthreads();

    // ---- coarse states.  Warp w owns the chunks [w cpw, (w+1) cpw) of 32 outputs.  The median rank of
    // the window of its first chunk comes from the count table; the following ones by sliding the
    // window 32 bins at a time: two ballots count the ranks under m that left and entered, and the
    // warp moves m by that many window elements, 32 places of the sorted order per step.
    const int n_coarse = (n_out + MED_PB - 1) / MED_PB;
    const int cpw = (n_coarse + WARPS - 1) / WARPS;
    const int c_first = warp * cpw;
    // warp-cooperative search: from rank wm (exclusive) in direction wdir to the wneed-th element whose
    // position lies in [wplo, wphi]; all arguments warp-uniform; wm is updated
#define WARP_SEEK(wm, wdir, wneed, wplo, wphi)                                                     \
        for (;;) {                                                                                 \
            const int r_ = (wm) + (wdir) * (1 + lane);                                             \
            const bool ok_ = (unsigned)r_ < (unsigned)LTe;                                         \
            const bool in_ = ok_ && (unsigned)((int)spos[ok_ ? r_ : 0] - (wplo)) <= (unsigned)((wphi) - (wplo)); \
            const unsigned bal_ = __ballot_sync(FULL, in_);                                        \
            const int cn_ = __popc(bal_);                                                          \
            if ((wneed) <= cn_) { (wm) += (wdir) * (1 + nth_set_bit(bal_, (wneed))); break; }      \
            (wneed) -= cn_;                                                                        \
            (wm) += 32 * (wdir);                                                                   \
            if ((unsigned)(wm) >= (unsigned)LTe) break;    /* not reachable: the window holds the element */ \
        }
    if (c_first < n_coarse) {
        int m = LTe;
        {
            const int c = c_first;
            const int j0 = c * MED_PB;
            const int b0 = c, b1 = (j0 + W) / MED_PB;
            const int na = b1 * MED_PB - j0;                 // block-aligned part of the window
            int below = 0, phi = j0 - 1;
            if (na > 0) {
                const int t = (h < na - 1) ? h : na - 1;
                // largest bucket lo with #{rank < 128 lo, position in the aligned part} <= t
                // (a bucket past the tile's last one counts everything: never chosen)
                const int c0 = lane < nrb ? (int)tab[lane * MED_TROW + b1] - (int)tab[lane * MED_TROW + b0] : 0x7fffffff;
                const int c1 = lane + 32 < nrb ? (int)tab[(lane + 32) * MED_TROW + b1] - (int)tab[(lane + 32) * MED_TROW + b0] : 0x7fffffff;
                const unsigned m0 = __ballot_sync(FULL, c0 <= t), m1 = __ballot_sync(FULL, c1 <= t);
                const int lo = m1 ? 63 - __clz(m1) : 31 - __clz(m0);
                const int cl = lo < 32 ? __shfl_sync(FULL, c0, lo & 31) : __shfl_sync(FULL, c1, lo & 31);
                int need = t - cl + 1;                       // the (t - cl + 1)-th aligned element from rank 128 lo on
                m = lo * MED_RB - 1;
                WARP_SEEK(m, 1, need, j0, j0 + na - 1);
                below = t;
                phi = b1 * MED_PB - 1;
            }
            // complete the window with the (at most 31, or W when W < 32) remaining positions
            for (int pbase = phi + 1; pbase < j0 + W; pbase += 32) {
                const int p = pbase + lane;
                const bool add = p < j0 + W && (int)rop[p < j0 + W ? p : 0] < m;
                below += __popc(__ballot_sync(FULL, add));
            }
            if (below > h) {                                 // down to the (below - h)-th window element under m
                int need = below - h;
                WARP_SEEK(m, -1, need, j0, j0 + W - 1);
            } else {                                         // up to the (h - below + 1)-th window element at or above m
                int need = h - below + 1;
                m -= 1;
                WARP_SEEK(m, 1, need, j0, j0 + W - 1);
            }
            if (lane == 0) cm[c] = (uint16_t)m;
        }
        const int c_last = (c_first + cpw < n_coarse) ? c_first + cpw : n_coarse;
        for (int c = c_first + 1; c < c_last; ++c) {
            const int j0 = c * MED_PB;                       // window [j0, j0 + W); the last one started 32 bins earlier
            const int gone = rop[j0 - MED_PB + lane], come = rop[j0 - MED_PB + W + lane];
            const int n_gone = __popc(__ballot_sync(FULL, gone < m)), n_come = __popc(__ballot_sync(FULL, come < m));
            const bool m_left = __ballot_sync(FULL, gone == m) != 0u;
            const int below = h + n_come - n_gone;
            int dir, need;
            if (below > h) { dir = -1; need = below - h; }
            else { dir = 1; need = h - below + (m_left ? 1 : 0); }
            if (need) { WARP_SEEK(m, dir, need, j0, j0 + W - 1); }
            if (lane == 0) cm[c] = (uint16_t)m;
        }
    }
    __syncthreads();                                         // the count table is dead from here on: orank may be written

    // ---- every thread walks MED_FINE outputs at a time, starting from the coarse state of its chunk.
    // `below` = #{window elements of rank < m}.  One rule for every move: the median is the
    // (below - h)-th window element under m, or the (h - below)-th above it, counting m itself first
    // when it is still in the window.  A thread steps along the sorted order on its own for at most
    // MED_STEP_CAP places; spectra with plateaus (wide chirps put the same power in consecutive bins)
    // and level-correlated neighbourhoods have stretches of hundreds of out-of-window elements, and
    // those searches are finished by the whole warp, 32 places per step.
    const int n_tasks = n_coarse * (MED_PB / MED_FINE);
    for (int task0 = 0; task0 < n_tasks; task0 += THREADS) {
        const int task = task0 + tid;
        const int s = task / n_coarse, c = task - s * n_coarse;
        const int j_first = c * MED_PB + s * MED_FINE;
        const bool alive = task < n_tasks && j_first < n_out;
        const int j_end = alive ? ((j_first + MED_FINE < n_out) ? j_first + MED_FINE : n_out) : j_first;
        int m = 0, plo = 0, phi = -1, dir = 1, need = 0;
#define IN_SET(r) ((unsigned)((int)spos[r] - plo) <= (unsigned)(phi - plo))
        // the warp completes the searches its lanes left unfinished: lane `src` still needs `need`
        // window elements from rank m (exclusive) in direction dir
#define WARP_FINISH()                                                                              \
        for (unsigned pend = __ballot_sync(FULL, need > 0); pend; pend &= pend - 1) {              \
            const int src = __ffs(pend) - 1;                                                       \
            int wm = __shfl_sync(FULL, m, src);                                                    \
            const int wdir = __shfl_sync(FULL, dir, src);                                          \
            int wneed = __shfl_sync(FULL, need, src);                                              \
            const int wplo = __shfl_sync(FULL, plo, src), wphi = __shfl_sync(FULL, phi, src);      \
            WARP_SEEK(wm, wdir, wneed, wplo, wphi);                                                \
            if (lane == src) { m = wm; need = 0; }                                                 \
        }
        if (alive) {
            int below = h;
            m = cm[c];
            plo = c * MED_PB;
            phi = plo + W - 1;
            // jump: count the ranks under m that left and entered
            const int jump = s * MED_FINE;
            for (int i = 0; i < jump; ++i) {
                below += ((int)rop[phi + 1 + i] < m) - ((int)rop[plo + i] < m);
            }
            plo += jump;
            phi += jump;
            if (below > h) { dir = -1; need = below - h; }
            else { dir = 1; need = h - below + (IN_SET(m) ? 0 : 1); }
            for (int t = 0; need && t < 3 * MED_STEP_CAP; ++t) { m += dir; if (IN_SET(m)) --need; }
        }
        WARP_FINISH();
        if (alive) orank[j_first] = (uint16_t)m;             // orank shares its memory with nothing the walk reads
#pragma unroll 1
        for (int jj = 1; jj < MED_FINE; ++jj) {
            const int j = j_first + jj;
            const bool on = j < j_end;
            if (on) {
                const int gone = rop[plo];                    // position j-1 leaves
                ++plo;
                const int come = rop[phi + 1];                // position j+2h enters
                ++phi;
                const int b = h + (come < m) - (gone < m);    // h-1, h or h+1
                dir = b > h ? -1 : 1;
                need = (b != h || gone == m) ? 1 : 0;
                for (int t = 0; need && t < MED_STEP_CAP; ++t) { m += dir; if (IN_SET(m)) need = 0; }
            }
            WARP_FINISH();
            if (on) orank[j] = (uint16_t)m;
        }
#undef WARP_FINISH
#undef IN_SET
    }
#undef WARP_SEEK
    __syncthreads();

    // ---- coalesced epilogue: median and PSD
    if (a.items && tid == 0) next_item = (int)gridDim.x + atomicAdd(&a.ctr[1], 1);
    double dmax = 0.0;
    for (int j0 = tid; j0 < n_out; j0 += 4 * THREADS) {
        double si[4];
        if (a.psd) {
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const int j = j0 + u * THREADS;
                si[u] = j < n_out ? __ldg(a.s_instr + o0 + j) : 0.0;
            }
        }
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const int j = j0 + u * THREADS;
            if (j < n_out) {
                int64_t v;
                if (NARROW) v = (int64_t)(((key_ref & 0xffffffff00000000ull) | (uint64_t)skey[orank[j]]) ^ SIGN64);
                else v = (int64_t)((uint64_t)skey[orank[j]] ^ SIGN64);
                const int64_t g = o0 + j;
                a.med[row + g] = v;
                neg |= v < 0;
                if (a.psd) {
                    const double e = (double)v * a.scale;
                    const double pnew = si[u] + a.norm * e;
                    if (DELTA) {                             // convergence in S_n: change against the last pass
                        const double pold = a.psd[row + g];
                        const double d = fabs(pnew - pold) / pold;
                        if (d > dmax) dmax = d;
                    }
                    a.psd[row + g] = pnew;
                }
            }
        }
    }
    if (DELTA) {                                         // non-negative binary64 values order like their bits
        for (int o = 16; o; o >>= 1) dmax = fmax(dmax, __shfl_xor_sync(FULL, dmax, o));
        if (lane == 0 && dmax > 0.0) atomicMax(a.delta_bits + row_i, (unsigned long long)__double_as_longlong(dmax));
    }
  }   // tiles
    if (a.neg_flag && neg) *a.neg_flag = 1;
}

}  // namespace gbfg
