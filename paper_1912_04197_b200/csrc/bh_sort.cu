// bh_sort.cu — step a3: stable LSD radix sort of (63-bit key, 32-bit body index), 8-bit digits.
// One kernel per digit pass ("onesweep" shape): each block takes a tile by atomic ticket, ranks its
// keys per warp with match.any ballots (stable: item order then lane order = index order), resolves
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
// chain (load, rank, look-back, two scatters), not bandwidth, sets a pass's time.  Measured (eight passes):
// 131072 keys 0.117 -> 0.085 ms with 2048-key tiles; 1M keys 0.171 ms with 4096-key tiles against 0.189 ms.
template <bool FIRST, int ITEMS>
__global__ void __launch_bounds__(kSortThreads, ITEMS == 16 ? 4 : 6)
sort_pass_kernel(const unsigned long long *__restrict__ kin, const unsigned *__restrict__ vin,
                 unsigned long long *__restrict__ kout, unsigned *__restrict__ vout, long long n, int shift,
                 const unsigned *__restrict__ hist, unsigned *lookback, unsigned *ticket)
{
    __shared__ unsigned long long skey[(kSortThreads * ITEMS)];          // 32 KB, reused for the values
    __shared__ unsigned whist[kSortThreads / 32][kRadix];   // per-warp digit counts -> offsets
    __shared__ unsigned sbase[kRadix];                      // global position of a digit's run - its tile offset
    __shared__ unsigned stoff[kRadix];                      // tile-local start of a digit's run
    __shared__ unsigned stmp[8];
    __shared__ unsigned stile;

    const unsigned tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
    if (tid == 0) stile = atomicAdd(ticket, 1u);
#pragma unroll
    for (int w = 0; w < kSortThreads / 32; ++w) whist[w][tid] = 0u;
    __syncthreads();
    const unsigned tile = stile;
    const long long base = (long long)tile * (kSortThreads * ITEMS);

    unsigned long long k[ITEMS];
    unsigned v[ITEMS];
    unsigned pos[ITEMS];
#pragma unroll
    for (int i = 0; i < ITEMS; ++i) {
        long long idx = base + warp * (32 * ITEMS) + i * 32 + lane;
        bool valid = idx < n;
        k[i] = valid ? kin[idx] : ~0ull;
        v[i] = FIRST ? (unsigned)idx : (valid ? vin[idx] : 0u);
    }
    // per-warp stable ranking, one item row at a time
    const unsigned lt = (1u << lane) - 1u;
#pragma unroll
    for (int i = 0; i < ITEMS; ++i) {
        long long idx = base + warp * (32 * ITEMS) + i * 32 + lane;
        bool valid = idx < n;
        unsigned d = (unsigned)(k[i] >> shift) & (kRadix - 1);
        unsigned peers = __match_any_sync(0xffffffffu, valid ? d : (kRadix + lane));
        unsigned pre = valid ? whist[warp][d] : 0u;
        __syncwarp();
        if (valid && (peers & lt) == 0u) whist[warp][d] = pre + __popc(peers);
        __syncwarp();
        pos[i] = pre + __popc(peers & lt);
    }
    __syncthreads();
    // digit = tid: exclusive prefix over the warps, tile total
    unsigned tot = 0;
#pragma unroll
    for (int w = 0; w < kSortThreads / 32; ++w) {
        unsigned c = whist[w][tid];
        whist[w][tid] = tot;
        tot += c;
    }
    // decoupled look-back over earlier tiles for this digit
    unsigned *mine = lookback + (size_t)tile * kRadix + tid;
    unsigned excl = 0;
    if (tile == 0) {
        st_relaxed(mine, kFlagPre | tot);
    } else {
        st_relaxed(mine, kFlagAgg | tot);
        // kLook predecessors are read per round trip to the L2 (independent loads), not one: the tiles of a pass
        // all publish their aggregates at about the same time, and the walk back to the nearest inclusive prefix
        // would otherwise be a chain of O(sqrt(tiles)) dependent loads
        constexpr int kLook = 8;
        long long t = (long long)tile - 1;
        bool done = false;
        while (!done) {
            unsigned s[kLook];
#pragma unroll
            for (int b = 0; b < kLook; ++b) {
                const long long u = t - b;
                s[b] = u >= 0 ? ld_relaxed(lookback + (size_t)u * kRadix + tid) : kFlagPre;   // before tile 0: nothing
            }
            int used = 0;
#pragma unroll
            for (int b = 0; b < kLook; ++b) {
                if (done || used != b) continue;     // stop at the first word that is not published yet
                if ((s[b] >> 30) == 0u) continue;
                excl += s[b] & kValMask;
                ++used;
                if (s[b] & kFlagPre) done = true;
            }
            t -= used;
        }
        st_relaxed(mine, kFlagPre | (excl + tot));
    }
    unsigned toff = block_excl_scan_256(tot, stmp);
    unsigned gbase = block_excl_scan_256(hist[tid], stmp);
    stoff[tid] = toff;
    sbase[tid] = gbase + excl - toff;
    __syncthreads();
    // tile-local sorted order in shared memory
#pragma unroll
    for (int i = 0; i < ITEMS; ++i) {
        long long idx = base + warp * (32 * ITEMS) + i * 32 + lane;
        if (idx < n) {
            unsigned d = (unsigned)(k[i] >> shift) & (kRadix - 1);
            pos[i] += stoff[d] + whist[warp][d];
            skey[pos[i]] = k[i];
        }
    }
    __syncthreads();
    long long rem = n - base;
    const unsigned nvalid = rem < (kSortThreads * ITEMS) ? (unsigned)rem : (unsigned)(kSortThreads * ITEMS);
    unsigned gpos[ITEMS];
#pragma unroll
    for (int j = 0; j < ITEMS; ++j) {
        unsigned i2 = tid + j * kSortThreads;
        if (i2 < nvalid) {
            unsigned long long kk = skey[i2];
            gpos[j] = sbase[(unsigned)(kk >> shift) & (kRadix - 1)] + i2;
            kout[gpos[j]] = kk;
        }
    }
    __syncthreads();
    unsigned *sval = reinterpret_cast<unsigned *>(skey);
#pragma unroll
    for (int i = 0; i < ITEMS; ++i) {
        long long idx = base + warp * (32 * ITEMS) + i * 32 + lane;
        if (idx < n) sval[pos[i]] = v[i];
    }
    __syncthreads();
#pragma unroll
    for (int j = 0; j < ITEMS; ++j) {
        unsigned i2 = tid + j * kSortThreads;
        if (i2 < nvalid) vout[gpos[j]] = sval[i2];
    }
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
