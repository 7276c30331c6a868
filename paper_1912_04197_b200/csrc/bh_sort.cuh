// bh_sort.cuh — block-level pieces of step a3 shared by the onesweep passes (bh_sort.cu) and the one-block
// build of small body sets (bh_small.cu): a 256-thread exclusive scan and a stable LSD radix sort of up to
// 256 x ITEMS (key, index) pairs that never leaves registers and shared memory.
#pragma once
#include "bh_common.cuh"

namespace bh {

// exclusive scan of one value per thread over a 256-thread block; tmp is 8 words of shared memory
__device__ __forceinline__ unsigned block_excl_scan_256(unsigned v, unsigned *tmp)
{
    const unsigned lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
    unsigned inc = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        unsigned t = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= (unsigned)o) inc += t;
    }
    if (lane == 31) tmp[warp] = inc;
    __syncthreads();
    unsigned base = 0;
#pragma unroll
    for (int k = 0; k < 8; ++k)
        if ((unsigned)k < warp) base += tmp[k];
    __syncthreads();
    return base + inc - v;
}

// exclusive scan of one value per digit (threads 0..255 hold a digit each, the others pass 0) over a block of
// THREADS >= 256 threads; tmp is 8 words of shared memory
template <int THREADS>
__device__ __forceinline__ unsigned block_excl_scan_digits(unsigned v, unsigned *tmp)
{
    const unsigned lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
    unsigned inc = v;
    if (warp < 8) {
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            unsigned t = __shfl_up_sync(0xffffffffu, inc, o);
            if (lane >= (unsigned)o) inc += t;
        }
        if (lane == 31) tmp[warp] = inc;
    }
    __syncthreads();
    unsigned base = 0;
#pragma unroll
    for (int k = 0; k < 8; ++k)
        if ((unsigned)k < warp) base += tmp[k];
    __syncthreads();
    return base + inc - v;
}

// Lanes of the warp that carry the same digit as this lane, from one ballot per digit bit (valid lanes only; an
// invalid lane is alone).  match.any gives the same mask in one instruction, but on sm_100 the eight ballots are
// much the faster way: the sort passes took 171 -> 134 us at 1M keys and 455 -> 359 us at 4M with them (measured,
// round 2), and the ncu capture of the match.any version had half of a pass's stall samples on the instruction
// after the match.
__device__ __forceinline__ unsigned digit_peers(unsigned d, bool valid, unsigned lane)
{
    unsigned peers = __ballot_sync(0xffffffffu, valid);
#pragma unroll
    for (int b = 0; b < kRadixBits; ++b) {
        const bool bit = (d >> b) & 1u;
        const unsigned m = __ballot_sync(0xffffffffu, bit);
        peers &= bit ? m : ~m;
    }
    return valid ? peers : (1u << lane);
}

// Rank of a key among the keys of its warp that carry the same digit and came before it (earlier rows, then lower
// lanes: index order, so the sort is stable).  cnt[256] are the warp's own running digit counters.
__device__ __forceinline__ unsigned warp_rank(unsigned *cnt, unsigned d, bool valid, unsigned lane, unsigned lt)
{
    const unsigned peers = digit_peers(d, valid, lane);
    const unsigned pre = valid ? cnt[d] : 0u;
    __syncwarp();
    if (valid && (peers & lt) == 0u) cnt[d] = pre + __popc(peers);
    __syncwarp();
    return pre + __popc(peers & lt);
}

// All eight digit passes inside one block of THREADS threads (a step over a few thousand bodies is bound by the
// latency of its dependent launches, "for a low number of bodies the computational time is dominated
// by the octree creation").  Thread t holds items  idx = warp * 32 * ITEMS + i * 32 + lane  (i < ITEMS), before and
// after; padding keys ~0 sort last in every pass (all digits 255, after the real 255s: stable).  Per-warp
// ballot ranking as in the tiled passes: stable by construction (item order, then lane order = index order).
// skey: THREADS * ITEMS keys of shared memory (reused for the values); whist: [THREADS / 32][256]; stoff: [256];
// stmp: [8].
template <int ITEMS, int THREADS>
__device__ __forceinline__ void block_radix_sort(unsigned long long (&k)[ITEMS], unsigned (&v)[ITEMS],
                                                 unsigned long long *skey, unsigned (*whist)[kRadix], unsigned *stoff,
                                                 unsigned *stmp, int p0 = 0)
{
    constexpr int kWarps = THREADS / 32;
    const unsigned tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
    const unsigned lt = (1u << lane) - 1u;
    unsigned pos[ITEMS];
#pragma unroll 1
    for (int p = p0; p < kSortPasses; ++p) {     // digits p0 .. 7 (p0 = 3: the partial-key sort, see repair_keys)
        const int shift = p * kRadixBits;
        for (int q = tid; q < kWarps * kRadix; q += THREADS) (&whist[0][0])[q] = 0u;
        __syncthreads();
#pragma unroll
        for (int i = 0; i < ITEMS; ++i) {
            const unsigned d = (unsigned)(k[i] >> shift) & (kRadix - 1);
            pos[i] = warp_rank(whist[warp], d, true, lane, lt);
        }
        __syncthreads();
        unsigned tot = 0;
        if (tid < (unsigned)kRadix) {   // digit = tid: exclusive prefix over the warps, total
#pragma unroll 8
            for (int w = 0; w < kWarps; ++w) {
                const unsigned c = whist[w][tid];
                whist[w][tid] = tot;
                tot += c;
            }
        }
        const unsigned off = block_excl_scan_digits<THREADS>(tot, stmp);
        if (tid < (unsigned)kRadix) stoff[tid] = off;
        __syncthreads();
#pragma unroll
        for (int i = 0; i < ITEMS; ++i) {
            const unsigned d = (unsigned)(k[i] >> shift) & (kRadix - 1);
            pos[i] += stoff[d] + whist[warp][d];
            skey[pos[i]] = k[i];
        }
        __syncthreads();
#pragma unroll
        for (int i = 0; i < ITEMS; ++i) k[i] = skey[warp * (32 * ITEMS) + i * 32 + lane];
        __syncthreads();
        unsigned *sval = reinterpret_cast<unsigned *>(skey);
#pragma unroll
        for (int i = 0; i < ITEMS; ++i) sval[pos[i]] = v[i];
        __syncthreads();
#pragma unroll
        for (int i = 0; i < ITEMS; ++i) v[i] = sval[warp * (32 * ITEMS) + i * 32 + lane];
        __syncthreads();
    }
}

// ---- one tile of a streaming digit pass (bh_sort.cu; also called by the one-kernel build of mid-size sets, bh_mid.cu) ----
constexpr unsigned kFlagAgg = 1u << 30;      // tile aggregate available
constexpr unsigned kFlagPre = 2u << 30;      // inclusive prefix available
constexpr unsigned kValMask = (1u << 30) - 1u;

__device__ __forceinline__ unsigned ld_relaxed(const unsigned *p)
{
    unsigned v;
    asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_relaxed(unsigned *p, unsigned v)
{
    asm volatile("st.relaxed.gpu.global.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}

// ITEMS keys per thread: 16 (tiles of 4096 keys, four blocks per SM at 64 registers) from 512k keys up; 8 (tiles of
// 2048 keys) below, where 4096-key tiles are too few to fill the machine and the length of one tile's dependent
// chain (load, rank, look-back, two scatters), not bandwidth, sets a pass's time.
// Order of a tile's work: load keys -> rank -> publish the tile's digit counts -> tile-local order of the keys in
// shared memory -> look back -> global scatter of keys, then of values.  The look-back comes as late as the data
// allow: the resident tiles of a pass publish their counts at about the same time, and the inclusive prefixes then
// travel down the tiles one look-back round at a time; whatever a tile can do without its global offsets it does
// while they travel.  A look-back round reads kLook predecessors at once (independent loads) and sleeps when it
// found nothing new, so that waiting tiles do not take issue slots from working ones (in the capture of round 2
// the spin was 37 % of a pass's instructions).  FULL tiles (all but the last) carry no bounds checks.
constexpr int kLook = 8;

// One round of look-back along a row array (stride kRadix words per row): reads up to kLook rows at once (independent
// loads), from row t downwards and not below row `floor`, adds the published ones in order and stops at the first
// unpublished one.  Returns the rows consumed; *pre is set once a row carried an inclusive prefix.
__device__ __forceinline__ int look_round(const unsigned *rows, long long t, long long floor, unsigned tid,
                                          unsigned &sum, bool &pre)
{
    unsigned s[kLook];
#pragma unroll
    for (int b = 0; b < kLook; ++b) s[b] = t - b >= floor ? ld_relaxed(rows + (size_t)(t - b) * kRadix + tid) : 0u;
    int used = 0;
#pragma unroll
    for (int b = 0; b < kLook; ++b) {
        if (pre || used != b || (s[b] >> 30) == 0u) continue;
        sum += s[b] & kValMask;
        ++used;
        if (s[b] & kFlagPre) pre = true;
    }
    return used;
}

// Exclusive prefix of this tile's digit count `tot` over all earlier tiles (decoupled look-back); publishes the
// tile's inclusive prefix.  look[tile][digit] holds a tile's own count (kFlagAgg) or its inclusive prefix (kFlagPre).
// Tiles are handed out in order by the ticket, so every row waited for belongs to a tile that is already running.
// (A second level of rows per group of 16 tiles, which shortens the walk of the first wave from ~12 to ~5 rounds,
// was built and measured in round 2: 130 -> 123 us at 1M keys but 338 -> 358 us at 4M and 1055 -> 1102 us at 16.7M,
// where the extra instructions cost more than the shorter walk saves; not kept.)
__device__ __forceinline__ unsigned look_back(unsigned *look, unsigned tile, unsigned tid, unsigned tot)
{
    if (tile == 0) return 0u;                                  // its count was published as an inclusive prefix
    unsigned excl = 0;
    bool pre = false;
    long long t = (long long)tile - 1;
    while (!pre) {
        const int used = look_round(look, t, 0, tid, excl, pre);
        t -= used;
        if (used == 0) __nanosleep(200);
    }
    st_relaxed(look + (size_t)tile * kRadix + tid, kFlagPre | (excl + tot));
    return excl;
}

template <bool FIRST, int ITEMS, bool FULL>
__device__ __forceinline__ void sort_tile(const unsigned long long *kin, const unsigned *vin,
                                          unsigned long long *kout, unsigned *vout,
                                          long long base, unsigned nvalid, unsigned tile, int shift,
                                          const unsigned *hist, unsigned *lookback,
                                          unsigned long long *skey, unsigned (*whist)[kRadix], unsigned *sbase,
                                          unsigned *stmp)
{
    const unsigned tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
    const unsigned woff = warp * (32 * ITEMS) + lane;     // item i of this thread is key woff + 32 i of the tile
    kin += base;
    unsigned long long k[ITEMS];
    unsigned pos[ITEMS];
#pragma unroll
    for (int i = 0; i < ITEMS; ++i) k[i] = (FULL || woff + 32 * i < nvalid) ? kin[woff + 32 * i] : ~0ull;
    // per-warp stable ranking, one item row at a time
    const unsigned lt = (1u << lane) - 1u;
#pragma unroll
    for (int i = 0; i < ITEMS; ++i) {
        const bool valid = FULL || woff + 32 * i < nvalid;
        const unsigned d = (unsigned)(k[i] >> shift) & (kRadix - 1);
        pos[i] = warp_rank(whist[warp], d, valid, lane, lt);
    }
    __syncthreads();
    // digit = tid: tile total (published at once), then the tile-local start of every (warp, digit) run
    unsigned tot = 0;
#pragma unroll
    for (int w = 0; w < kSortThreads / 32; ++w) tot += whist[w][tid];
    unsigned *mine = lookback + (size_t)tile * kRadix + tid;
    st_relaxed(mine, (tile == 0 ? kFlagPre : kFlagAgg) | tot);
    const unsigned toff = block_excl_scan_256(tot, stmp);
    {
        unsigned run = toff;
#pragma unroll
        for (int w = 0; w < kSortThreads / 32; ++w) {
            const unsigned c = whist[w][tid];
            whist[w][tid] = run;
            run += c;
        }
    }
    __syncthreads();
    // tile-local sorted order of the keys in shared memory
#pragma unroll
    for (int i = 0; i < ITEMS; ++i) {
        if (FULL || woff + 32 * i < nvalid) {
            const unsigned d = (unsigned)(k[i] >> shift) & (kRadix - 1);
            pos[i] += whist[warp][d];
            skey[pos[i]] = k[i];
        }
    }
    // the values are requested before the look-back, so that they arrive while it waits
    unsigned v[ITEMS];
    if (!FIRST) {
        vin += base;
#pragma unroll
        for (int i = 0; i < ITEMS; ++i) v[i] = (FULL || woff + 32 * i < nvalid) ? vin[woff + 32 * i] : 0u;
    } else {
#pragma unroll
        for (int i = 0; i < ITEMS; ++i) v[i] = (unsigned)base + woff + 32 * i;
    }
    // decoupled look-back over earlier tiles for this digit
    const unsigned excl = look_back(lookback, tile, tid, tot);
    const unsigned gbase = block_excl_scan_256(hist[tid], stmp);
    sbase[tid] = gbase + excl - toff;
    __syncthreads();
    unsigned gpos[ITEMS];
#pragma unroll
    for (int j = 0; j < ITEMS; ++j) {
        const unsigned i2 = tid + j * kSortThreads;
        if (FULL || i2 < nvalid) {
            const unsigned long long kk = skey[i2];
            gpos[j] = sbase[(unsigned)(kk >> shift) & (kRadix - 1)] + i2;
            kout[gpos[j]] = kk;
        }
    }
    __syncthreads();
    unsigned *sval = reinterpret_cast<unsigned *>(skey);
#pragma unroll
    for (int i = 0; i < ITEMS; ++i)
        if (FULL || woff + 32 * i < nvalid) sval[pos[i]] = v[i];
    __syncthreads();
#pragma unroll
    for (int j = 0; j < ITEMS; ++j) {
        const unsigned i2 = tid + j * kSortThreads;
        if (FULL || i2 < nvalid) vout[gpos[j]] = sval[i2];
    }
}

// ---- the repair pass of the partial-key sort (bh_sort.cu; also a phase of the one-kernel build, bh_mid.cu) ----
constexpr int kHighFirst = 3;                // first digit of the partial sort: digits 3..7 = key bits 24..63
constexpr int kLowBits = kHighFirst * kRadixBits;
constexpr unsigned kRunMax = 64;             // longest run the quadratic repair takes
constexpr int kRepairPer = 4;                // keys per thread of the repair pass, their loads issued together

// kRepairPer keys j0, j0 + 256, ... of an array that is stably sorted by its top 39 bits: each goes to its place in the
// order by the full key (ties by position).  Returns true if a run was longer than kRunMax (nothing is written for it).
__device__ __forceinline__ bool repair_keys(const unsigned long long *kin, const unsigned *vin, unsigned long long *kout,
                                            unsigned *vout, long long n, long long j0)
{
    unsigned long long k[kRepairPer], kl[kRepairPer], kr[kRepairPer];
    unsigned v[kRepairPer];
#pragma unroll
    for (int u = 0; u < kRepairPer; ++u) {
        const long long j = j0 + (long long)u * kSortThreads;
        const bool in = j < n;
        k[u] = in ? kin[j] : 0ull;
        v[u] = in ? vin[j] : 0u;
        kl[u] = (in && j > 0) ? kin[j - 1] : ~0ull;          // ~0 >> 24 is no valid top: keys have 63 bits
        kr[u] = (in && j + 1 < n) ? kin[j + 1] : ~0ull;
    }
    bool too_long = false;
#pragma unroll
    for (int u = 0; u < kRepairPer; ++u) {
        const long long j = j0 + (long long)u * kSortThreads;
        if (j >= n) continue;
        const unsigned long long top = k[u] >> kLowBits;
        if ((kl[u] >> kLowBits) != top && (kr[u] >> kLowBits) != top) {   // alone in its run (the usual case): it stays
            kout[j] = k[u];
            vout[j] = v[u];
            continue;
        }
        long long lo = j, hi = j + 1;        // the run is [lo, hi)
        while (lo > 0 && j - lo <= (long long)kRunMax && (kin[lo - 1] >> kLowBits) == top) --lo;
        while (hi < n && hi - j <= (long long)kRunMax && (kin[hi] >> kLowBits) == top) ++hi;
        if (hi - lo > (long long)kRunMax) {
            too_long = true;
            continue;
        }
        long long r = lo;
        for (long long i = lo; i < hi; ++i) {
            const unsigned long long ki = kin[i];
            r += (ki < k[u]) || (ki == k[u] && i < j);
        }
        kout[r] = k[u];
        vout[r] = v[u];
    }
    return too_long;
}

}  // namespace bh
