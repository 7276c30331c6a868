// bh_sort.cu — step a3: stable LSD radix sort of (63-bit key, 32-bit body index), 8-bit digits.
// One kernel per digit pass ("onesweep" shape): each block takes a tile by atomic ticket, ranks its
// keys per warp with one ballot per digit bit (stable: item order then lane order = index order), resolves
// the tile's global digit offsets with a decoupled look-back over the tiles before it, and scatters
// through shared memory so that the global writes are runs of consecutive addresses per digit.
// The global digit histograms of all passes were accumulated by keys_kernel.
#include "bh_sort.cuh"

namespace bh {

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
__device__ __forceinline__ void sort_tile(const unsigned long long *__restrict__ kin, const unsigned *__restrict__ vin,
                                          unsigned long long *__restrict__ kout, unsigned *__restrict__ vout,
                                          long long base, unsigned nvalid, unsigned tile, int shift,
                                          const unsigned *__restrict__ hist, unsigned *lookback,
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

template <bool FIRST, int ITEMS>
__global__ void __launch_bounds__(kSortThreads, ITEMS == 16 ? 3 : 5)
sort_pass_kernel(const unsigned long long *__restrict__ kin, const unsigned *__restrict__ vin,
                 unsigned long long *__restrict__ kout, unsigned *__restrict__ vout, long long n, int shift,
                 const unsigned *__restrict__ hist, unsigned *lookback, unsigned *ticket)
{
    __shared__ unsigned long long skey[(kSortThreads * ITEMS)];          // 32 KB, reused for the values
    __shared__ unsigned whist[kSortThreads / 32][kRadix];   // per-warp digit counts -> tile-local starts of the (warp, digit) runs
    __shared__ unsigned sbase[kRadix];                      // global position of a digit's run - its tile offset
    __shared__ unsigned stmp[8];
    __shared__ unsigned stile;

    const unsigned tid = threadIdx.x;
    if (tid == 0) stile = atomicAdd(ticket, 1u);
#pragma unroll
    for (int w = 0; w < kSortThreads / 32; ++w) whist[w][tid] = 0u;
    __syncthreads();
    const unsigned tile = stile;
    const long long base = (long long)tile * (kSortThreads * ITEMS);
    const long long rem = n - base;
    if (rem >= kSortThreads * ITEMS)
        sort_tile<FIRST, ITEMS, true>(kin, vin, kout, vout, base, (unsigned)(kSortThreads * ITEMS), tile, shift, hist,
                                      lookback, skey, whist, sbase, stmp);
    else
        sort_tile<FIRST, ITEMS, false>(kin, vin, kout, vout, base, (unsigned)rem, tile, shift, hist, lookback, skey,
                                       whist, sbase, stmp);
}

// keys per tile of the streaming passes for n keys
int sort_tile_items(int64_t n) { return n < kSortSmallTileBelow ? 8 : 16; }

int launch_sort(const Workspace &w, int64_t n, cudaStream_t s)
{
    const int items = sort_tile_items(n);
    const int tiles = (int)((n + kSortThreads * items - 1) / (kSortThreads * items));
    for (int p = 0; p < kSortPasses; ++p) {
        const int a = p & 1, b = a ^ 1;
        unsigned *lb = w.lookback + (size_t)p * tiles * kRadix;   // [pass][tiles of this n][256]: cleared per build
#define BH_SORT_PASS(FIRST, ITEMS)                                                                                     \
    sort_pass_kernel<FIRST, ITEMS><<<tiles, kSortThreads, 0, s>>>(w.key[a], w.idx[a], w.key[b], w.idx[b], n,           \
                                                                  p * kRadixBits, w.hist + p * kRadix, lb, w.sort_ticket + p)
        if (items == 8) {
            if (p == 0) BH_SORT_PASS(true, 8);
            else BH_SORT_PASS(false, 8);
        } else {
            if (p == 0) BH_SORT_PASS(true, 16);
            else BH_SORT_PASS(false, 16);
        }
#undef BH_SORT_PASS
    }
    return kSortPasses;
}

}  // namespace bh
