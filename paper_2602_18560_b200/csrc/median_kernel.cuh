// median_kernel.cuh — the running-median tile kernel (stage iii), included by median.cu.
//
// running_median_tile_kernel<KeyT, THREADS>:
//   <uint32_t, 512>   the fast variant: two CTAs per SM, so that one tile's sort overlaps the other's
//                     walk (every phase of the tile loop is bound by shared-memory latency and barriers,
//                     not by issue slots).  Keys are the low 32 bits of the biased spectrum values, which
//                     order a tile whenever its values agree in their high 32 bits — spectra in units of
//                     2^-140 strain^2 always do.  A tile that does not is appended to the wide list.
//   <uint64_t, 1024>  full 64-bit keys, one CTA per SM: the tiles of the wide list.
// See median.cu for the algorithm (sort once per tile, window bitmaps over the sorted order, word-wise walk).
#pragma once

#include "gbfg_common.cuh"

namespace gbfg {

// Positions per tile, halos included.  32-bit keys: 17 x 512; with W = 2001 a tile then holds up to 6704 outputs and a full
// row of the 4-yr grid (3 774 349 bins) is 592 tiles = exactly two tiles for each of the 296 resident CTAs (8192 positions
// made it 888 = three each, with a third more positions sorted per output).  64-bit keys: the next multiple of 1024.
constexpr int MED_LT32 = 8704;
constexpr int MED_LT64 = 9216;
constexpr int MED_PB = 32;                    // outputs per chunk (one per lane)
#ifndef MED_MLP
#define MED_MLP 4                             // global loads a thread keeps in flight while it stages a tile / writes it out
#endif
#ifndef MED_MATCH_EVERY
#define MED_MATCH_EVERY 3                     // sort rounds whose peer masks come from MATCH.ANY: one in this many
#endif
constexpr int MED_CROW = 256 + 2;             // radix counter row stride in u16 (one row per warp)
constexpr uint64_t SIGN64 = 0x8000000000000000ull;

// aux: the radix counters (one row per warp) during the sort; afterwards one window bitmap per warp (LT bits) and,
// behind them, the output ranks
__host__ __device__ constexpr int median_aux_u16(int threads, int lt)
{
    const int warps = threads / 32;
    const int sort_u16 = warps * MED_CROW;
    const int walk_u16 = 2 * warps * (lt / 32 + 1) * 2;               // window and specials bitmaps, rows of lt / 32 + 1 words
    return sort_u16 > walk_u16 ? sort_u16 : walk_u16;
}

template <typename KeyT, int THREADS, int LT>
constexpr size_t median_smem_bytes()
{
    return sizeof(KeyT) * LT                              // skey
         + sizeof(uint16_t) * LT                          // spos
         + sizeof(uint16_t) * LT                          // rop
         + sizeof(uint16_t) * median_aux_u16(THREADS, LT) // radix counters, then the window bitmaps
         + sizeof(uint32_t) * 40;                         // scan partials, varying-bit mask
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
#ifdef MED_TIMING
    long long *dbg;          // probe builds only (-DMED_TIMING): [gridDim.x][16] cycles per phase, summed over a CTA's tiles
#endif
};

#ifdef MED_TIMING
// phase i = the time between tick i and the tick before it, summed over the CTA's tiles, per CTA
#define MED_TICK(i) do { if (tid == 0) { const long long now_ = clock64(); if (i) a.dbg[blockIdx.x * 16 + (i)] += now_ - med_t_prev; med_t_prev = now_; } } while (0)
// inside the sort: the time since the last sub-tick, summed over the passes
#define MED_SUBTICK(i) do { if (tid == 0) { const long long now_ = clock64(); a.dbg[blockIdx.x * 16 + (i)] += now_ - med_t_sub; med_t_sub = now_; } } while (0)
#else
#define MED_TICK(i) do { } while (0)
#define MED_SUBTICK(i) do { } while (0)
#endif

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

// bit updates of the window bitmaps: shared-memory reductions on a 32-bit shared address (the generic-address form
// costs a dozen instructions of address arithmetic per update)
__device__ __forceinline__ void smem_or(uint32_t addr, unsigned v)
{
    asm volatile("red.shared.or.b32 [%0], %1;" ::"r"(addr), "r"(v) : "memory");
}
__device__ __forceinline__ void smem_and(uint32_t addr, unsigned v)
{
    asm volatile("red.shared.and.b32 [%0], %1;" ::"r"(addr), "r"(v) : "memory");
}

// loads from a 32-bit shared address (the arrays of the tile sit at constant offsets from one base: no generic
// pointers to keep, no 64-bit address arithmetic in the walk)
__device__ __forceinline__ unsigned smem_ld32(uint32_t addr)
{
    unsigned v;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(addr) : "memory");
    return v;
}
__device__ __forceinline__ unsigned smem_ld16(uint32_t addr)
{
    unsigned short v;
    asm volatile("ld.shared.u16 %0, [%1];" : "=h"(v) : "r"(addr) : "memory");
    return v;
}

// lanes of the warp whose 8-bit digit equals this lane's: what match.any computes, from 8 ballots.  MATCH.ANY is a
// single instruction but the SM retires only one every ~50 clocks (measured: a radix pass over 8192 keys takes 19 000
// clocks with it, 12 700 with the ballots, and two CTAs on one SM no longer slow each other down)
__device__ __forceinline__ unsigned same_digit_lanes(unsigned d)
{
    unsigned peers = 0xffffffffu;
    const unsigned me = 1u << (threadIdx.x & 31);
#pragma unroll
    for (int b = 0; b < 8; ++b) {
        const unsigned sb = (unsigned)((int)(d << (31 - b)) >> 31);            // all ones when bit b of the digit is set
        const unsigned bal = __reduce_or_sync(0xffffffffu, me & sb);           // a ballot; REDUX retires a little faster than VOTE here
        peers &= ~(bal ^ sb);                                                  // bit set: & bal, clear: & ~bal
    }
    return peers;
}

// 32 x 32 bit matrix, row i in lane i -> column j in lane j (bit i of the result of lane j = bit j of the value of
// lane i): five butterfly steps, each one shuffle
template <int K, unsigned M>
__device__ __forceinline__ unsigned transpose_bits_step(unsigned v, int lane)
{
    const unsigned x = __shfl_xor_sync(0xffffffffu, v, K);
    const bool upper = lane & K;
    const unsigned xs = upper ? (x >> K) : (x << K);
    const unsigned take = upper ? M : ~M;                                      // the bits that come from the partner
    return (v & ~take) | (xs & take);
}
__device__ __forceinline__ unsigned transpose_bits_32(unsigned v)
{
    const int lane = threadIdx.x & 31;
    v = transpose_bits_step<16, 0x0000ffffu>(v, lane);
    v = transpose_bits_step<8, 0x00ff00ffu>(v, lane);
    v = transpose_bits_step<4, 0x0f0f0f0fu>(v, lane);
    v = transpose_bits_step<2, 0x33333333u>(v, lane);
    v = transpose_bits_step<1, 0x55555555u>(v, lane);
    return v;
}

// DELTA: also record the largest relative PSD change (the second stop rule, R13); a template parameter so
// that the default kernel carries none of it
template <typename KeyT, int THREADS, int LT, bool DELTA>
__global__ void __launch_bounds__(THREADS, THREADS <= 512 ? 2 : 1)
running_median_tile_kernel(MedianArgs a)
{
    constexpr int WARPS = THREADS / 32;
    constexpr int ITEMS = (LT + THREADS - 1) / THREADS;   // keys per thread in the sort, at most
    static_assert(LT % THREADS == 0 && LT % 32 == 0 && LT <= 65536, "tile size");
    constexpr int GROUPS = WARPS / 8;                      // counter scan: thread t owns digit t / GROUPS, 8 warps
    constexpr bool NARROW = sizeof(KeyT) == 4;
    static_assert(THREADS == 256 * GROUPS, "the counter scan maps one thread to one (digit, 8 warps) group");

    extern __shared__ __align__(16) unsigned char smem_raw[];
    KeyT *skey = reinterpret_cast<KeyT *>(smem_raw);
    uint16_t *spos = reinterpret_cast<uint16_t *>(skey + LT);
    uint16_t *rop = spos + LT;
    uint16_t *aux = rop + LT;                          // radix counters; then the window bitmaps and the output ranks
    constexpr int AUX_U16 = median_aux_u16(THREADS, LT);
    uint32_t *misc = reinterpret_cast<uint32_t *>(aux + AUX_U16);
    uint32_t *aux32 = reinterpret_cast<uint32_t *>(aux);

    const int tid = threadIdx.x;
    const int warp = tid >> 5, lane = tid & 31;
    const unsigned FULL = 0xffffffffu;
    const unsigned lt_mask = (1u << lane) - 1u;
    const int h = a.h, W = 2 * a.h + 1;
    __shared__ int s_item;
#ifdef MED_TIMING
    long long med_t_prev = 0, med_t_sub = 0;
#endif
    int flags = 0;                                       // bit 0: a negative median (kernel-wide); bit 1: a median on a saturated key (this tile)
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
    const int rounds = (Lt + THREADS - 1) / THREADS;
    const int LTe = rounds * THREADS;                    // positions sorted

    MED_TICK(0);
    // ---- stage the tile: position p <-> global bin o0 - h + p, reflected at both ends.
    // Unused positions (Lt <= p < LTe) repeat position 0: they are never inside a window.
    if (tid < 5) misc[32 + tid] = tid == 2 ? 0xffffffffu : 0u;      // varying bits (lo, hi), smallest high word, varying bits again, keys >= 2^24
    __syncthreads();
    uint64_t key_ref;
    {
        int64_t g0 = o0 - h;
        if (g0 < 0) g0 = -g0 - 1;
        if (g0 >= a.n) g0 = 2 * a.n - 1 - g0;
        key_ref = (uint64_t)a.x[row + g0] ^ SIGN64;
        uint64_t vary = 0;
        for (int p0 = tid; p0 < LTe; p0 += MED_MLP * THREADS) {    // MED_MLP independent loads in flight per thread
            uint64_t key[MED_MLP];
#pragma unroll
            for (int u = 0; u < MED_MLP; ++u) {
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
            for (int u = 0; u < MED_MLP; ++u) {
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
    uint64_t vary_all = ((uint64_t)misc[33] << 32) | misc[32];
    bool saturated = false;                              // keys above the tile's smallest high word share the key 0xffffffff
    if (NARROW && (vary_all >> 32) != 0) {
        // 32 bits do not order this tile.  Most often a handful of very loud bins stick out above 2^32 while the medians
        // sit far below: every value whose high word exceeds the tile's smallest one then gets the key 0xffffffff (they
        // are all larger than the rest, and their order among themselves does not matter as long as no median is one of
        // them, which the walk checks).  Otherwise, or when that check fails, the tile goes to the 64-bit-key kernel.
        // (Not with the PSD-change rule: a second attempt would compare against the first attempt's PSD.)
        if (DELTA) {
            if (tid == 0) {
                a.wide_items[atomicAdd(&a.wide_ctr[0], 1)] = make_int4(row_i, (int)o0, n_out, 0);
                if (a.items) next_item = (int)gridDim.x + atomicAdd(&a.ctr[1], 1);
            }
            continue;
        }
        unsigned hmin = 0xffffffffu;
        for (int p = tid; p < Lt; p += THREADS) {
            int64_t g = o0 - h + p;
            if (g < 0) g = -g - 1;
            if (g >= a.n) g = 2 * a.n - 1 - g;
            const unsigned hi = (unsigned)(((uint64_t)__ldg(a.x + row + g) ^ SIGN64) >> 32);
            hmin = hi < hmin ? hi : hmin;
        }
        hmin = __reduce_min_sync(FULL, hmin);
        if (lane == 0) atomicMin(&misc[34], hmin);
        __syncthreads();
        hmin = misc[34];
        const unsigned k_first = (unsigned)(key_ref >> 32) == hmin ? (unsigned)key_ref : 0xffffffffu;
        unsigned vary32 = 0u;
        for (int p = tid; p < LTe; p += THREADS) {
            unsigned k32 = k_first;
            if (p < Lt) {
                int64_t g = o0 - h + p;
                if (g < 0) g = -g - 1;
                if (g >= a.n) g = 2 * a.n - 1 - g;
                const uint64_t key = (uint64_t)__ldg(a.x + row + g) ^ SIGN64;
                k32 = (unsigned)(key >> 32) == hmin ? (unsigned)key : 0xffffffffu;
            }
            vary32 |= k32 ^ k_first;
            skey[p] = (KeyT)k32;
        }
        vary32 = __reduce_or_sync(FULL, vary32);
        if (lane == 0 && vary32) atomicOr(&misc[35], vary32);
        __syncthreads();
        vary_all = misc[35];
        key_ref = ((uint64_t)hmin << 32) | k_first;      // the high word of every value that can be a median
        saturated = true;
    }
    int n_pass = vary_all ? (64 - __clzll((long long)vary_all) + 7) / 8 : 0;
    if (NARROW && n_pass == 4) {
        // A fourth pass only for a few loud bins: with no more than h keys at or above 2^24 in the tile no window can have
        // one of them as its median (a window of 2h+1 then holds at least h+1 smaller ones), so they may all become the
        // largest 24-bit key: the ranks below them stay exact, and three passes sort the tile.
        int big = 0;
        for (int p = tid; p < LTe; p += THREADS) big += (unsigned)skey[p] >= 0x01000000u;
        big = __reduce_add_sync(FULL, big);
        if (lane == 0 && big) atomicAdd(&misc[36], (unsigned)big);
        __syncthreads();
        if (misc[36] <= (unsigned)h) {
            for (int p = tid; p < LTe; p += THREADS)
                if ((unsigned)skey[p] >= 0x01000000u) skey[p] = (KeyT)0x00ffffffu;
            __syncthreads();
            n_pass = 3;
        }
    }

    MED_TICK(1);
    // ---- LSD radix sort by key, stable, so that equal keys stay in position order.
    // Warp w owns elements [32 rounds w, 32 rounds (w + 1)) of the current order, 32 consecutive ones per round.
    for (int pass = 0; pass < n_pass; ++pass) {
        const int shift = 8 * pass;
#ifdef MED_TIMING
        if (tid == 0) med_t_sub = clock64();
#endif
        for (int e = tid; e < WARPS * MED_CROW / 2; e += THREADS) aux32[e] = 0u;
        __syncthreads();
        MED_SUBTICK(8);
        uint16_t *cw = aux + warp * MED_CROW;
        KeyT k[ITEMS];
        uint32_t pk[ITEMS];                              // position << 16 | place among the warp's keys of the same digit
#pragma unroll
        for (int r = 0; r < ITEMS; ++r) {                // the matches are independent: issue them together
            if (r < rounds) {
                const int e = warp * (32 * rounds) + r * 32 + lane;
                k[r] = skey[e];
                // every third round by MATCH.ANY, the others by eight reductions: the two run on different units of the
                // SM (one MATCH per ~50 clocks, ~50 issue slots for the reductions), so the mix beats either alone
                pk[r] = (r % MED_MATCH_EVERY == 0) ? __match_any_sync(FULL, (unsigned)(k[r] >> shift) & 255u)
                                     : same_digit_lanes((unsigned)(k[r] >> shift) & 255u);
            }
        }
        MED_SUBTICK(9);
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
        MED_SUBTICK(10);
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
        MED_SUBTICK(11);
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
        MED_SUBTICK(12);
    }

    MED_TICK(2);
    // ---- inverse permutation: rop[p] = rank of position p
    for (int r = tid; r < LTe; r += THREADS) rop[spos[r]] = (uint16_t)r;
    __syncthreads();

    MED_TICK(3);
    if (a.items && tid == 0) next_item = (int)gridDim.x + atomicAdd(&a.ctr[1], 1);     // the next tile of this CTA
    double dmax = 0.0;
    flags &= 1;
    // ---- window bitmaps.  Warp w owns the chunks [w cpw, (w+1) cpw) of 32 consecutive outputs and keeps, in
    // shared memory, one bit per sorted rank: "the element of this rank lies in the window".  The median of a
    // window is its (h+1)-th set bit.
    //  * The bitmaps of the warps' first windows are built by the whole CTA from the rank side (a bit transpose per
    //    two words of ranks, below), no read-modify-write; each warp then finds its first median by counting words.
    //  * Inside a chunk lane i takes output j0 + i.  The 32 positions that leave and the 32 that enter while the
    //    window slides over the chunk are the chunk's "specials" (a second bitmap marks their ranks); every other
    //    set bit of U = window(j0) + the entering positions lies in all the chunk's windows.  Two popcounts of
    //    ballots tell lane i how many elements of its own window it has to move from the chunk's first median m0,
    //    and in which direction; it then moves word by word (32 ranks and, typically, 8 window elements per step:
    //    a popcount), looking at positions only for the specials of a word, and picks the bit inside the last
    //    word.  Lane 0, whose own answer is m0, does the same for output j0 + 32: the first median of the next
    //    chunk.  Plateaus and long stretches of out-of-window ranks cost one step per 32 ranks.
    {
        const int n_coarse = (n_out + MED_PB - 1) / MED_PB;
        const int cpw = (n_coarse + WARPS - 1) / WARPS;
        const int c_first = warp * cpw;
        const int c_last = (c_first + cpw < n_coarse) ? c_first + cpw : n_coarse;
        constexpr int BMW = LT / 32 + 1;                         // words per bitmap row (odd: rows start on different banks)
        unsigned *bm = aux32 + warp * BMW;
        unsigned *sp = aux32 + (WARPS + warp) * BMW;
        const int nw = LTe / 32;
        // (kept opaque to the compiler: it would otherwise work the address out again from the CTA's shared window and the
        // warp index in every round of the walk, nine instructions, rather than hold it in a register)
        uint32_t bm_a = (uint32_t)__cvta_generic_to_shared(bm);
        asm volatile("" : "+r"(bm_a));
        {
            // Position p lies in the first window of warp w2 iff w2 wstep <= p < w2 wstep + W (wstep = the outputs of a
            // warp): a range of w2, i.e. a mask of at most 32 bits per lane.  What warp w2 needs is the transposed thing,
            // for every word of 32 ranks the lanes whose mask has bit w2: one 32 x 32 bit transpose per word (sixteen
            // warps: per two words, their 16-bit masks side by side) instead of one ballot per (word, warp).
            const int wstep = cpw * MED_PB;
            const int n_chain = (n_coarse + cpw - 1) / cpw;      // warps that have a chunk
            const unsigned magic = 0xffffffffu / (unsigned)wstep + 1u;     // p / wstep = umulhi(p, magic) for p wstep < 2^32
            const int back = wstep - W;
            auto first_windows = [&](int p) -> unsigned {
                const unsigned hi = min(__umulhi((unsigned)p, magic), 31u);
                const unsigned lo = __umulhi((unsigned)max(p + back, 0), magic);
                return lo > hi ? 0u : (((2u << hi) - 1u) & ~((1u << lo) - 1u));
            };
            if (WARPS == 16) {
                // nw is a multiple of 16: lanes 0-15 get word e2 for the warps 0-15, lanes 16-31 word e2 + 1
                for (int e2 = 2 * warp; e2 < nw; e2 += 2 * WARPS) {
                    const int pa = spos[(e2 << 5) + lane], pb = spos[((e2 + 1) << 5) + lane];
                    const unsigned v = transpose_bits_32((first_windows(pa) & 0xffffu) | (first_windows(pb) << 16));
                    if ((lane & 15) < n_chain) aux32[(lane & 15) * BMW + e2 + (lane >> 4)] = v;
                }
            } else {
                for (int e = warp; e < nw; e += WARPS) {
                    const unsigned v = transpose_bits_32(first_windows(spos[(e << 5) + lane]));
                    if (lane < n_chain) aux32[lane * BMW + e] = v;
                }
            }
            for (int e = lane; e < nw; e += 32) sp[e] = 0u;
        }
        __syncthreads();
        MED_TICK(4);
        if (c_first < c_last) {
            int j0 = c_first * MED_PB;
            int m0;
            {   // the (h+1)-th set bit: lane l counts the words [l per, (l+1) per)
                const int per = (nw + 31) / 32;
                int cnt = 0;
                for (int q = 0; q < per; ++q) { const int e = lane * per + q; cnt += e < nw ? __popc(bm[e]) : 0; }
                int incl = cnt;
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) {
                    const int up = __shfl_up_sync(FULL, incl, o);
                    if (lane >= o) incl += up;
                }
                const unsigned reach = __ballot_sync(FULL, incl >= h + 1);
                const int L = __ffs(reach) - 1;
                int found = 0;
                if (lane == L) {
                    int need = h + 1 - (incl - cnt);              // 1-based among this lane's words
                    for (int q = 0; q < per; ++q) {
                        const int e = lane * per + q;
                        const unsigned wd = e < nw ? bm[e] : 0u;
                        const int pc = __popc(wd);
                        if (need <= pc) { found = e * 32 + nth_set_bit(wd, need); break; }
                        need -= pc;
                    }
                }
                m0 = __shfl_sync(FULL, found, L);
            }
            MED_TICK(5);
            // the arrays as 32-bit shared addresses: skey at 0, spos, rop, then the bitmaps (sp of a warp SP_D behind its bm)
            uint32_t sm0 = (uint32_t)__cvta_generic_to_shared(smem_raw);
            asm volatile("" : "+r"(sm0));
            constexpr uint32_t SPOS_A = sizeof(KeyT) * LT, ROP_A = SPOS_A + 2u * LT, SP_D = 4u * WARPS * BMW;
            int64_t *const med_row = a.med + row + o0;           // output j of the tile: med_row[j]
            double *const psd_row = a.psd ? a.psd + row + o0 : nullptr;
            const double *const si_row = a.s_instr ? a.s_instr + o0 : nullptr;
            for (int c = c_first; c < c_last; ++c, j0 += MED_PB) {
                const int pg = j0 + lane, pc_ = j0 + W + lane;           // positions that leave / enter
                // this lane's own output is j0 + lane: what its PSD needs is on its way while the median is found
                const bool own = pg < n_out;
                double si = 0.0, pold = 0.0;
                if (psd_row && own) {
                    si = __ldg(si_row + pg);
                    if (DELTA) pold = psd_row[pg];
                }
                const int gone = (int)smem_ld16(sm0 + ROP_A + 2u * (uint32_t)pg);
                const bool c_ok = pc_ < Lt;
                const int come = c_ok ? (int)smem_ld16(sm0 + ROP_A + 2u * (uint32_t)pc_) : 0x7fffffff;
                const unsigned gb = __ballot_sync(FULL, gone < m0), cb = __ballot_sync(FULL, come < m0);
                const unsigned gm = __ballot_sync(FULL, gone == m0);
                const uint32_t g_off = (uint32_t)(gone >> 5) << 2, c_off = (uint32_t)(come >> 5) << 2;
                const unsigned g_bit = 1u << (gone & 31), c_bit = 1u << (come & 31);
                smem_or(bm_a + SP_D + g_off, g_bit);
                if (c_ok) {
                    smem_or(bm_a + c_off, c_bit);
                    smem_or(bm_a + SP_D + c_off, c_bit);
                }
                // lane i: output j0 + i; lane 0: output j0 + 32 (the next chunk's first), its own answer being m0
                const bool next_needed = c + 1 < c_last;
                const int i_eff = lane ? lane : 32;
                const unsigned before = lane ? lt_mask : FULL;            // the slides k < i_eff
                const int delta = __popc(cb & before) - __popc(gb & before);
                const bool present = (gm & before) == 0u;
                int t;
                bool up;
                if (delta > 0) { up = false; t = delta; }
                else { up = true; t = -delta + (present ? 0 : 1); }
                const int jlo = j0 + i_eff;
                if (lane ? (jlo >= n_out) : !next_needed) t = 0;
                __syncwarp();
                int r = m0;
                // the word the lane's answer lies in, and which of its bits (from below or from above) it is; the bit itself
                // is picked once for the whole warp behind the loop (inside it, lanes that end in different rounds would
                // each run the search on their own)
                unsigned w_fin = 1u;
                int t_fin = 1, wi = m0 >> 5;
                bool moved = false;
                if (t > 0) {
                    const int step = up ? 1 : -1;
                    // the first word: only the ranks beyond m0
                    unsigned keep = up ? ~((2u << (m0 & 31)) - 1u) : ((1u << (m0 & 31)) - 1u);
                    for (;;) {
                        const uint32_t w_a = bm_a + 4u * (uint32_t)wi;
                        unsigned wb = smem_ld32(w_a) & keep;
                        for (unsigned sb = wb & smem_ld32(w_a + SP_D); sb; sb &= sb - 1u) {       // specials: in this lane's window?
                            const int b = __ffs(sb) - 1;
                            const int pos = (int)smem_ld16(sm0 + SPOS_A + 2u * (uint32_t)((wi << 5) + b));
                            if ((unsigned)(pos - jlo) >= (unsigned)W) wb &= ~(1u << b);
                        }
                        const int pc = __popc(wb);
                        if (t <= pc) { w_fin = wb; t_fin = t; moved = true; break; }
                        t -= pc;
                        wi += step;
                        keep = 0xffffffffu;
                        if ((unsigned)wi >= (unsigned)nw) break;               // not reachable: the window holds the element
                    }
                }
                {
                    // the t-th set bit from below (up) or from above (down): one search, on the word or its mirror image
                    const int at = nth_set_bit(up ? w_fin : __brev(w_fin), t_fin);
                    if (moved) r = (wi << 5) + (up ? at : 31 - at);
                }
                if (own) {                                   // median and PSD of output j0 + lane, 256 bytes per warp and array
                    const int at = lane ? r : m0;
                    KeyT kv;
                    if (NARROW) kv = (KeyT)smem_ld32(sm0 + 4u * (uint32_t)at);
                    else kv = skey[at];
                    if (NARROW && saturated && kv == (KeyT)0xffffffffu) flags |= 2;
                    int64_t v;
                    if (NARROW) v = (int64_t)(((key_ref & 0xffffffff00000000ull) | (uint64_t)kv) ^ SIGN64);
                    else v = (int64_t)((uint64_t)kv ^ SIGN64);
                    med_row[pg] = v;
                    flags |= (int)(v < 0);
                    if (psd_row) {
                        const double e = (double)v * a.scale;
                        const double pnew = si + a.norm * e;
                        if (DELTA) {                         // convergence in S_n: change against the last pass
                            const double d = fabs(pnew - pold) / pold;
                            if (d > dmax) dmax = d;
                        }
                        psd_row[pg] = pnew;
                    }
                }
                __syncwarp();
                smem_and(bm_a + g_off, ~g_bit);
                smem_and(bm_a + SP_D + g_off, ~g_bit);
                if (c_ok) smem_and(bm_a + SP_D + c_off, ~c_bit);
                m0 = __shfl_sync(FULL, r, 0);
                __syncwarp();
            }
        }
    }
    {
        const int any_hit = __syncthreads_or(NARROW && saturated && (flags & 2));      // (also the barrier of the walk's end)
        if (NARROW && any_hit && tid == 0) a.wide_items[atomicAdd(&a.wide_ctr[0], 1)] = make_int4(row_i, (int)o0, n_out, 0);
    }

    MED_TICK(6);
    if (DELTA) {                                         // non-negative binary64 values order like their bits
        for (int o = 16; o; o >>= 1) dmax = fmax(dmax, __shfl_xor_sync(FULL, dmax, o));
        if (lane == 0 && dmax > 0.0) atomicMax(a.delta_bits + row_i, (unsigned long long)__double_as_longlong(dmax));
    }
    MED_TICK(7);
  }   // tiles
    if (a.neg_flag && (flags & 1)) *a.neg_flag = 1;
}

}  // namespace gbfg
