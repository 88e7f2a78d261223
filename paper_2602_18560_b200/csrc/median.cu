// median.cu — stage (iii): exact running median of eq. (D2) + the PSD of eq. (10).
//
// DESIGN.md R3: odd window W = 2h+1 centred on k, ends reflected, statistic = the h-th smallest
// of the 2h+1 int64 values.  Only integer comparisons decide the result, so it is exact.
//
// Persistent CTAs, one per SM, take tiles of at most S = LT - 2h consecutive outputs — from the work
// list plan_kernel derives from the blocks the last subtraction made dirty, or (stage call) from a
// static tiling of every row.  The tile and its two h-bin halos (Lt = outputs + 2h <= LT positions,
// rounded up to a multiple of 1024) are
// staged in shared memory and sorted ONCE by (value, position): an LSD radix sort, 8 bits per pass,
// that skips the passes whose digit is the same for the whole tile (spectrum values rarely need
// more than four).  With the sorted order in hand a window is a position interval, and its median
// is found without ever sorting a window:
//   * a (rank-bucket x position-block) table of counts locates the h-th smallest element of a
//     block-aligned position interval; one warp does this for the start of every chunk of 32
//     outputs (coarse states);
//   * every thread then takes 8 outputs: it jumps from the coarse state to its first output by
//     counting the ranks that left and entered, and walks: sliding the window by one bin removes
//     one position and adds one, which moves the median by at most one place in the sorted order;
//     the neighbouring in-window element is found by stepping through the sorted positions
//     (on average LT/W steps).
// The per-output rank is kept in shared memory and written out coalesced, fused with
//     psd[k] = s_instr[k] + C * (med[k] * 2^scale_log2)        (eqs. 10, D2, D3).
#include "gbfg_common.cuh"

namespace gbfg {

constexpr int MED_LT = 8192;                  // positions per tile, halos included (power of two)
constexpr int MED_THREADS = 1024;
constexpr int MED_WARPS = MED_THREADS / 32;
constexpr int MED_ITEMS = MED_LT / MED_THREADS;   // 8 keys per thread in the sort
constexpr int MED_PB = 32;                    // position block = outputs per coarse chunk
constexpr int MED_FINE = 8;                   // outputs per walking thread
constexpr int MED_STEP_CAP = 12;               // places a thread steps alone before the warp takes over
constexpr int MED_RB = 128;                   // sorted ranks per bucket
constexpr int MED_NPB = MED_LT / MED_PB;      // 256
constexpr int MED_NRB = MED_LT / MED_RB;      // 64
constexpr int MED_TROW = MED_NPB + 2;         // table row stride in u16 (even: rows stay 4-byte aligned)
constexpr int MED_CROW = 256 + 2;             // radix counter row stride in u16 (one row per warp)
constexpr uint64_t SIGN64 = 0x8000000000000000ull;

constexpr size_t MED_AUX_U16 = (MED_NRB * MED_TROW > MED_WARPS * MED_CROW) ? MED_NRB * MED_TROW : MED_WARPS * MED_CROW;
constexpr size_t MED_SMEM = sizeof(uint64_t) * MED_LT      // skey
                          + sizeof(uint16_t) * MED_LT      // spos
                          + sizeof(uint16_t) * MED_LT      // rop
                          + sizeof(uint16_t) * MED_LT      // orank
                          + sizeof(uint16_t) * MED_AUX_U16 // radix counters, then the count table
                          + sizeof(uint16_t) * MED_NPB     // coarse medians
                          + sizeof(uint32_t) * 40;         // scan partials, varying-bit mask

struct MedianArgs {
    const int64_t *x;        // [n_cat][n]
    int64_t *med;            // [n_cat][n]
    const double *s_instr;   // [n] or NULL (no PSD)
    double *psd;             // [n_cat][n] or NULL
    const int4 *items;       // work list (row, first output, outputs, -) or NULL: static tiling of every row
    int *ctr;                // [0] number of items, [1] next item
    int n_cat;
    int *neg_flag;           // nullable: set to 1 when a median is negative
    int64_t n;
    int h;
    int S;                   // outputs per tile = MED_LT - 2h
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

__global__ void __launch_bounds__(MED_THREADS, 1)
running_median_kernel(MedianArgs a)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    uint64_t *skey = reinterpret_cast<uint64_t *>(smem_raw);
    uint16_t *spos = reinterpret_cast<uint16_t *>(skey + MED_LT);
    uint16_t *rop = spos + MED_LT;
    uint16_t *orank = rop + MED_LT;
    uint16_t *aux = orank + MED_LT;                       // radix counters, later the count table
    uint16_t *cm = aux + MED_AUX_U16;                     // coarse medians
    uint32_t *misc = reinterpret_cast<uint32_t *>(cm + MED_NPB);
    uint16_t *tab = aux;
    uint32_t *aux32 = reinterpret_cast<uint32_t *>(aux);

    const int tid = threadIdx.x;
    const int warp = tid >> 5, lane = tid & 31;
    const unsigned FULL = 0xffffffffu;
    const unsigned lt_mask = (1u << lane) - 1u;
    const int h = a.h, W = 2 * a.h + 1;
    __shared__ int s_item;
    bool neg = false;

  for (int64_t turn = blockIdx.x;; turn += gridDim.x) {
    int64_t row, o0;
    int n_out;
    __syncthreads();                                     // the previous tile's epilogue is done with shared memory
    if (a.items) {
        if (tid == 0) s_item = atomicAdd(&a.ctr[1], 1);
        __syncthreads();
        const int item = s_item;
        if (item >= a.ctr[0]) break;
        const int4 v = a.items[item];
        row = (int64_t)v.x * a.n;
        o0 = v.y;
        n_out = v.z;
    } else {
        if (turn >= (int64_t)a.tiles * a.n_cat) break;
        const int64_t r = turn / a.tiles, tile = turn - r * a.tiles;
        row = r * a.n;
        o0 = tile * a.S;
        n_out = (int)((a.n - o0 < a.S) ? (a.n - o0) : a.S);
    }
    const int Lt = n_out + 2 * h;                        // positions really used
    const int rounds = (Lt + MED_THREADS - 1) / MED_THREADS;   // keys per thread in the sort (<= MED_ITEMS)
    const int LTe = rounds * MED_THREADS;                // positions sorted

    // ---- stage the tile: position p <-> global bin o0 - h + p, reflected at both ends.
    // Unused positions (Lt <= p < LTe) repeat position 0: they are never inside a window.
    if (tid < 2) misc[32 + tid] = 0u;
    __syncthreads();
    {
        int64_t g0 = o0 - h;
        if (g0 < 0) g0 = -g0 - 1;
        if (g0 >= a.n) g0 = 2 * a.n - 1 - g0;
        const uint64_t key_ref = (uint64_t)a.x[row + g0] ^ SIGN64;
        uint64_t vary = 0;
        for (int p = tid; p < LTe; p += MED_THREADS) {
            uint64_t key = key_ref;
            if (p < Lt) {
                int64_t g = o0 - h + p;
                if (g < 0) g = -g - 1;
                if (g >= a.n) g = 2 * a.n - 1 - g;
                key = (uint64_t)a.x[row + g] ^ SIGN64;
            }
            vary |= key ^ key_ref;
            skey[p] = key;
            spos[p] = (uint16_t)p;
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
    const int n_pass = vary_all ? (64 - __clzll((long long)vary_all) + 7) / 8 : 0;

    // ---- LSD radix sort by key, stable, so that equal keys stay in position order.
    // Warp w owns elements [32 rounds w, 32 rounds (w + 1)) of the current order, 32 consecutive ones per round.
    for (int pass = 0; pass < n_pass; ++pass) {
        const int shift = 8 * pass;
        for (int e = tid; e < MED_WARPS * MED_CROW / 2; e += MED_THREADS) aux32[e] = 0u;
        __syncthreads();
        uint16_t *cw = aux + warp * MED_CROW;
        uint64_t k[MED_ITEMS];
        uint32_t pp[MED_ITEMS], off[MED_ITEMS], peers[MED_ITEMS];
#pragma unroll
        for (int r = 0; r < MED_ITEMS; ++r) {            // the matches are independent: issue them together
            if (r < rounds) {
                const int e = warp * (32 * rounds) + r * 32 + lane;
                k[r] = skey[e];
                pp[r] = spos[e];
                off[r] = (unsigned)(k[r] >> shift) & 255u;
                peers[r] = same_digit_lanes(off[r]);
            }
        }
#pragma unroll
        for (int r = 0; r < MED_ITEMS; ++r) {            // counter updates, round after round
            if (r < rounds) {
                const unsigned d = off[r];
                const unsigned base = cw[d];
                __syncwarp();
                const unsigned rank = __popc(peers[r] & lt_mask);
                if (rank == 0) cw[d] = (uint16_t)(base + __popc(peers[r]));
                __syncwarp();
                off[r] = (d << 16) | (base + rank);
            }
        }
        __syncthreads();
        {   // exclusive scan of the counters in (digit, warp) order: thread t owns digit t/4, warps 8(t%4)..+8
            const int d = tid >> 2, wg = (tid & 3) * 8;
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
            unsigned wt = misc[lane], wincl = wt;
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
        for (int r = 0; r < MED_ITEMS; ++r) {
            if (r < rounds) {
                const unsigned dst = (unsigned)cw[off[r] >> 16] + (off[r] & 0xffffu);
                skey[dst] = k[r];
                spos[dst] = (uint16_t)pp[r];
            }
        }
        __syncthreads();
    }

    // ---- inverse permutation and the count table
    for (int e = tid; e < MED_NRB * MED_TROW / 2; e += MED_THREADS) aux32[e] = 0u;
    __syncthreads();
    for (int r = tid; r < LTe; r += MED_THREADS) {
        int p = spos[r];
        rop[p] = (uint16_t)r;
        int e = (r / MED_RB) * MED_TROW + (p / MED_PB) + 1;
        atomicAdd(&aux32[e >> 1], (e & 1) ? 0x10000u : 1u);
    }
    __syncthreads();
    // prefix along the position blocks: tab[rb][pb] = #{r in bucket rb : pos < pb*PB}
    {
        constexpr int PER = (MED_NPB + 1 + 31) / 32;     // 9 entries per lane
        for (int rb = warp; rb < MED_NRB; rb += MED_WARPS) {
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
                int up = __shfl_up_sync(FULL, incl, o);
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

    // ---- coarse states.  Warp w owns the chunks [w cpw, (w+1) cpw) of 32 outputs.  The median rank of
    // the window of its first chunk comes from the count table; the following ones by sliding the
    // window 32 bins at a time: two ballots count the ranks under m that left and entered, and the
    // warp moves m by that many window elements, 32 places of the sorted order per step.
    const int n_coarse = (n_out + MED_PB - 1) / MED_PB;
    const int cpw = (n_coarse + MED_WARPS - 1) / MED_WARPS;
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
                const int c0 = (int)tab[lane * MED_TROW + b1] - (int)tab[lane * MED_TROW + b0];
                const int c1 = (int)tab[(lane + 32) * MED_TROW + b1] - (int)tab[(lane + 32) * MED_TROW + b0];
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
    __syncthreads();

    // ---- every thread walks MED_FINE outputs, starting from the coarse state of its chunk.
    // `below` = #{window elements of rank < m}.  One rule for every move: the median is the
    // (below - h)-th window element under m, or the (h - below)-th above it, counting m itself first
    // when it is still in the window.  A thread steps along the sorted order on its own for at most
    // MED_STEP_CAP places; spectra with plateaus (wide chirps put the same power in consecutive bins)
    // and level-correlated neighbourhoods have stretches of hundreds of out-of-window elements, and
    // those searches are finished by the whole warp, 32 places per step.
    {
        const int s = tid / n_coarse, c = tid - s * n_coarse;
        const int j_first = c * MED_PB + s * MED_FINE;
        const bool alive = s < MED_PB / MED_FINE && j_first < n_out;
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
        if (alive) orank[j_first] = (uint16_t)m;
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
#undef WARP_SEEK
#undef IN_SET
    }
    __syncthreads();

    // ---- coalesced epilogue: median and PSD
    for (int j = tid; j < n_out; j += MED_THREADS) {
        int64_t v = (int64_t)(skey[orank[j]] ^ SIGN64);
        int64_t g = o0 + j;
        a.med[row + g] = v;
        neg |= v < 0;
        if (a.psd) {
            double e = (double)v * a.scale;
            a.psd[row + g] = a.s_instr[g] + a.norm * e;
        }
    }
  }   // tiles
    if (a.neg_flag && neg) *a.neg_flag = 1;
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

// ---------------------------------------------------------------------------------------------
// plan_kernel: one CTA per row.  Turns the dirty-block stamps of the last subtraction into
//   cum[row][b]  = number of dirty blocks before block b (b = 0 .. n_dblk), and
//   the work list of the running median: every maximal run of dirty blocks is cut into pieces of at
//   most S outputs (runs longer than one wave of CTAs are cut into a multiple of `wave` pieces).
// all_dirty != 0: every block counts as dirty (first iteration, cap branch without tracking).
// ctr[0] must be zero on entry; ctr[1] (the consumers' ticket) likewise.
// ---------------------------------------------------------------------------------------------
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
};

// len < 2^31 (n_bins is): 32-bit divisions, the 64-bit ones are long instruction sequences
static size_t plan_smem_bytes(int n_dblk) { return sizeof(int) * (size_t)((n_dblk + 1) + 3 * (n_dblk / 2 + 1)); }

__device__ __forceinline__ void plan_pieces(int64_t len64, int S, int wave, int *pieces, int *piece_len)
{
    const unsigned len = (unsigned)len64;
    unsigned np = (len + (unsigned)S - 1u) / (unsigned)S;
    if (np > (unsigned)wave) np = (np + (unsigned)wave - 1u) / (unsigned)wave * (unsigned)wave;
    const unsigned pl = (len + np - 1u) / np;
    *piece_len = (int)pl;
    *pieces = (int)((len + pl - 1u) / pl);
}

__global__ void __launch_bounds__(PLAN_THREADS)
plan_kernel(PlanArgs a)
{
    extern __shared__ int s_cum[];                      // [n_dblk + 1], then the runs: 3 ints each, [n_dblk / 2 + 1]
    __shared__ int wtot[32];
    __shared__ int n_runs, row_pieces, row_base;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int row = blockIdx.x;
    const int nb = a.n_dblk;
    const int *st = a.blk_stamp ? a.blk_stamp + (int64_t)row * nb : nullptr;
    int *cum = a.cum + (int64_t)row * (nb + 1);
    const int per = (nb + PLAN_THREADS - 1) / PLAN_THREADS;
    const int b_lo = min(tid * per, nb), b_hi = min(b_lo + per, nb);
    int *s_run = s_cum + nb + 1;
    if (tid == 0) { n_runs = 0; row_pieces = 0; }
    if (row == 0 && a.zero_ptr) for (int i = tid; i < a.zero_n; i += PLAN_THREADS) a.zero_ptr[i] = 0;
    for (int b0 = tid; b0 < nb; b0 += 8 * PLAN_THREADS) {   // coalesced, eight loads in flight per thread
        int v[8];
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            const int b = b0 + u * PLAN_THREADS;
            v[u] = (!a.all_dirty && b < nb) ? st[b] : a.stamp;
        }
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            const int b = b0 + u * PLAN_THREADS;
            if (b < nb) s_cum[b + 1] = (v[u] == a.stamp) ? 1 : 0;
        }
    }
    __syncthreads();
    int cnt = 0;
    for (int b = b_lo; b < b_hi; ++b) cnt += s_cum[b + 1];
    int incl = cnt;
    for (int o = 1; o < 32; o <<= 1) {
        const int up = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += up;
    }
    if (lane == 31) wtot[warp] = incl;
    __syncthreads();
    int run = incl - cnt;
    for (int w = 0; w < warp; ++w) run += wtot[w];
    if (tid == 0) s_cum[0] = 0;
    for (int b = b_lo; b < b_hi; ++b) {                 // s_cum[b + 1] = flag of block b -> inclusive count
        run += s_cum[b + 1];
        s_cum[b + 1] = run;
    }
    __syncthreads();
    for (int b = tid; b <= nb; b += PLAN_THREADS) {
        cum[b] = s_cum[b];
        if (b < nb && s_cum[b + 1] != s_cum[b]) {          // first / last dirty block of the row
            if (s_cum[b] == 0) a.range[2 * row] = b;
            if (s_cum[b + 1] == s_cum[nb]) a.range[2 * row + 1] = b;
        }
    }
    if (tid == 0 && s_cum[nb] == 0) { a.range[2 * row] = 1; a.range[2 * row + 1] = 0; }
    __syncthreads();
    // Tile size of this row: S outputs at most, less when the dirty part of the row would not fill
    // the row's share of one wave of CTAs (the latency of a short tile is what the tail iterations pay).
    int S = a.S;
    {
        const unsigned dirty_out = (unsigned)s_cum[nb] << a.dblk_log2;      // <= n_bins + one block
        int share = a.wave / (int)gridDim.x;
        if (share < 1) share = 1;
        unsigned s_fit = (dirty_out + (unsigned)share - 1u) / (unsigned)share;
        if (s_fit < (unsigned)PLAN_MIN_OUT) s_fit = PLAN_MIN_OUT;
        if (s_fit < (unsigned)S) S = (int)s_fit;
    }
    // runs: a dirty block whose predecessor is clean starts one; its end by bisection on cum.
    // Every run is recorded in shared memory with the place of its pieces in the row's part of the
    // list; then the warps write the items, one run per warp at a time.
    for (int b = b_lo; b < b_hi; ++b) {
        const bool dirty = s_cum[b + 1] != s_cum[b];
        if (!dirty || (b > 0 && s_cum[b] != s_cum[b - 1])) continue;
        int lo = b + 1, hi = nb;                        // largest e in [b+1, nb] with cum[e] - cum[b] == e - b
        while (lo < hi) {
            const int mid = (lo + hi + 1) >> 1;
            if (s_cum[mid] - s_cum[b] == mid - b) lo = mid; else hi = mid - 1;
        }
        const int e = lo;
        const int64_t first = (int64_t)b << a.dblk_log2;
        int64_t last = (int64_t)e << a.dblk_log2;
        if (last > a.n_bins) last = a.n_bins;
        int pieces, piece_len;
        plan_pieces(last - first, S, a.wave, &pieces, &piece_len);
        const int slot = atomicAdd(&n_runs, 1);
        s_run[3 * slot] = b;
        s_run[3 * slot + 1] = e;
        s_run[3 * slot + 2] = atomicAdd(&row_pieces, pieces);
    }
    __syncthreads();
    if (tid == 0) {
        if (a.out_count) {                               // dirty outputs of the row = dirty blocks, the last one clipped
            int64_t outs = (int64_t)s_cum[nb] << a.dblk_log2;
            if (nb > 0 && s_cum[nb] != s_cum[nb - 1]) outs -= ((int64_t)nb << a.dblk_log2) - a.n_bins;
            a.out_count[row] += outs;
        }
        if (gridDim.x == 1) { row_base = 0; a.ctr[0] = row_pieces; a.ctr[1] = 0; }
        else row_base = atomicAdd(&a.ctr[0], row_pieces);
    }
    __syncthreads();
    const int nr = n_runs, rb0 = row_base;
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
}

int median_tile_outputs(int window) { return MED_LT - (window - 1); }

int median_tiles(int64_t n_bins, int window)
{
    int S = MED_LT - (window - 1);
    return (int)((n_bins + S - 1) / S);
}

// upper bound of the number of work items plan_kernel can emit for one row
int median_max_items(int64_t n_bins)
{
    const int s_min = MED_LT - (GBFG_MAX_WINDOW - 1);
    const int s_small = s_min < PLAN_MIN_OUT ? s_min : PLAN_MIN_OUT;
    return dirty_blocks_per_row(n_bins) + 2 * (int)((n_bins + s_small - 1) / s_small) + 16;
}

// work list + cum from the stamps (blk_stamp NULL or all_dirty: everything)
int launch_plan(const int *blk_stamp, int stamp, bool all_dirty, int64_t n_bins, int n_cat, int window,
                const MedianPlan &pl, int64_t *zero_ptr, int zero_n, int64_t *out_count, cudaStream_t st)
{
    PlanArgs a;
    a.zero_ptr = zero_ptr; a.zero_n = zero_n; a.out_count = out_count;
    a.blk_stamp = blk_stamp; a.stamp = stamp; a.all_dirty = (all_dirty || !blk_stamp) ? 1 : 0;
    a.n_dblk = pl.n_dblk; a.dblk_log2 = pl.dblk_log2; a.n_bins = n_bins;
    a.S = MED_LT - (window - 1);
    a.wave = sm_count();
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
// launch_plan on the same stream); NULL: every row, statically tiled.  neg_flag nullable: raised when
// a median is negative.
int launch_median(const int64_t *x, int64_t n_bins, int n_cat, int window, int64_t *med,
                  const double *s_instr, double *psd, double norm, int scale_log2,
                  const MedianPlan *plan, int *neg_flag, cudaStream_t st)
{
    MedianArgs a;
    a.x = x; a.med = med; a.s_instr = s_instr; a.psd = psd; a.neg_flag = neg_flag;
    a.items = plan ? plan->items : nullptr; a.ctr = plan ? plan->ctr : nullptr; a.n_cat = n_cat;
    a.n = n_bins; a.h = window / 2;
    const int s_max = MED_LT - 2 * a.h;
    const int sms = sm_count();
    // static tiling: whole waves of CTAs when a row needs more than one
    int64_t tiles = (n_bins + s_max - 1) / s_max;
    if (tiles * n_cat > sms && n_cat == 1) tiles = (tiles + sms - 1) / sms * sms;
    a.S = (int)((n_bins + tiles - 1) / tiles);
    a.tiles = (int)((n_bins + a.S - 1) / a.S);
    a.norm = norm; a.scale = ldexp(1.0, scale_log2);
    static thread_local int attr_dev = -1;
    int dev = 0;
    GBFG_CUDA(cudaGetDevice(&dev));
    if (attr_dev != dev) {
        GBFG_CUDA(cudaFuncSetAttribute(running_median_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)MED_SMEM));
        attr_dev = dev;
    }
    int64_t grid = plan ? sms : (int64_t)a.tiles * n_cat;
    if (grid > sms) grid = sms;
    {
        LaunchTimer lt(K_MEDIAN, st);
        running_median_kernel<<<(int)grid, MED_THREADS, MED_SMEM, st>>>(a);
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
    return launch_median(dev_spectrum, n_bins, n_cat, window, dev_median_out, nullptr, nullptr, 1.0, 0, nullptr, nullptr,
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

