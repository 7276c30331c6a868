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

#ifndef BH_SORT_MINBLOCKS
#define BH_SORT_MINBLOCKS 4   // 64 registers (80 bytes spilled): four blocks per SM instead of two; sort at 4M bodies 0.60 -> 0.50 ms, 1M unchanged
#endif
template <bool FIRST>
__global__ void __launch_bounds__(kSortThreads, BH_SORT_MINBLOCKS)
sort_pass_kernel(const unsigned long long *__restrict__ kin, const unsigned *__restrict__ vin,
                 unsigned long long *__restrict__ kout, unsigned *__restrict__ vout, long long n, int shift,
                 const unsigned *__restrict__ hist, unsigned *lookback, unsigned *ticket)
{
    __shared__ unsigned long long skey[kSortTile];          // 32 KB, reused for the values
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
    const long long base = (long long)tile * kSortTile;

    unsigned long long k[kSortItems];
    unsigned v[kSortItems];
    unsigned pos[kSortItems];
#pragma unroll
    for (int i = 0; i < kSortItems; ++i) {
        long long idx = base + warp * (32 * kSortItems) + i * 32 + lane;
        bool valid = idx < n;
        k[i] = valid ? kin[idx] : ~0ull;
        v[i] = FIRST ? (unsigned)idx : (valid ? vin[idx] : 0u);
    }
    // per-warp stable ranking, one item row at a time
    const unsigned lt = (1u << lane) - 1u;
#pragma unroll
    for (int i = 0; i < kSortItems; ++i) {
        long long idx = base + warp * (32 * kSortItems) + i * 32 + lane;
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
        long long t = (long long)tile - 1;
        while (true) {
            unsigned s = ld_relaxed(lookback + (size_t)t * kRadix + tid);
            if ((s >> 30) == 0u) continue;   // not published yet
            excl += s & kValMask;
            if (s & kFlagPre) break;
            --t;
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
    for (int i = 0; i < kSortItems; ++i) {
        long long idx = base + warp * (32 * kSortItems) + i * 32 + lane;
        if (idx < n) {
            unsigned d = (unsigned)(k[i] >> shift) & (kRadix - 1);
            pos[i] += stoff[d] + whist[warp][d];
            skey[pos[i]] = k[i];
        }
    }
    __syncthreads();
    long long rem = n - base;
    const unsigned nvalid = rem < kSortTile ? (unsigned)rem : (unsigned)kSortTile;
    unsigned gpos[kSortItems];
#pragma unroll
    for (int j = 0; j < kSortItems; ++j) {
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
    for (int i = 0; i < kSortItems; ++i) {
        long long idx = base + warp * (32 * kSortItems) + i * 32 + lane;
        if (idx < n) sval[pos[i]] = v[i];
    }
    __syncthreads();
#pragma unroll
    for (int j = 0; j < kSortItems; ++j) {
        unsigned i2 = tid + j * kSortThreads;
        if (i2 < nvalid) vout[gpos[j]] = sval[i2];
    }
}

int launch_sort(const Workspace &w, int64_t n, cudaStream_t s)
{
    const int tiles = (int)((n + kSortTile - 1) / kSortTile);   // one tile: the whole build is one block (bh_small.cu)
    for (int p = 0; p < kSortPasses; ++p) {
        const int a = p & 1, b = a ^ 1;
        unsigned *lb = w.lookback + (size_t)p * tiles * kRadix;   // [pass][tiles of this n][256]: cleared per build
        if (p == 0)
            sort_pass_kernel<true><<<tiles, kSortThreads, 0, s>>>(w.key[a], w.idx[a], w.key[b], w.idx[b], n,
                                                                 p * kRadixBits, w.hist + p * kRadix, lb,
                                                                 w.sort_ticket + p);
        else
            sort_pass_kernel<false><<<tiles, kSortThreads, 0, s>>>(w.key[a], w.idx[a], w.key[b], w.idx[b], n,
                                                                  p * kRadixBits, w.hist + p * kRadix, lb,
                                                                  w.sort_ticket + p);
    }
    return kSortPasses;
}

}  // namespace bh
