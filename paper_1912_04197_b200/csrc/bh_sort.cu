// bh_sort.cu — step a3: stable LSD radix sort of (63-bit key, 32-bit body index), 8-bit digits.
// One kernel per digit pass ("onesweep" shape): each block takes a tile by atomic ticket, ranks its
// keys per warp with one ballot per digit bit (stable: item order then lane order = index order), resolves
// the tile's global digit offsets with a decoupled look-back over the tiles before it, and scatters
// through shared memory so that the global writes are runs of consecutive addresses per digit.
// The global digit histograms of all passes were accumulated by keys_kernel.
#include "bh_sort.cuh"

namespace bh {

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
