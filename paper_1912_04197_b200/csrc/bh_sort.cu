// bh_sort.cu — step a3: stable LSD radix sort of (63-bit key, 32-bit body index), 8-bit digits.
// One kernel per digit pass ("onesweep" shape): each block takes a tile by atomic ticket, ranks its
// keys per warp with one ballot per digit bit (stable: item order then lane order = index order), resolves
// the tile's global digit offsets with a decoupled look-back over the tiles before it, and scatters
// through shared memory so that the global writes are runs of consecutive addresses per digit.
// The global digit histograms of all passes were accumulated by keys_kernel.
#include <cstdlib>

#include "bh_keys.cuh"
#include "bh_sort.cuh"
#include "bh_grid.cuh"

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

// ------------------------------------------------------------------------------------------ partial-key sort
// Only the FIVE high digits (the top 39 key bits) go through digit passes.  Stable passes leave every run of keys with
// equal top bits in index order; a repair pass then ranks each key inside its run by (low 24 bits, position) and writes
// it to its final place.  Runs are short where bodies are distinct points (longest run 6 at configs[3], 2 at
// configs[4]: they are the bodies of one level-13 cell), so the repair is one more streaming pass without ranking
// machinery.  A run longer than kRunMax (coincident bodies share all 63 bits) raises a flag instead, and the last
// kernel of the sort — a co-resident grid that leaves at once when the flag is down — then sorts from scratch with all
// eight digits (grid barriers between the passes).  Either way the result is the stable order by the full key: the
// same permutation, bit for bit.  Five passes end in buffer 1, the repair moves the data to buffer 0.
__global__ void __launch_bounds__(kSortThreads)
sort_repair_kernel(const unsigned long long *__restrict__ kin, const unsigned *__restrict__ vin,
                   unsigned long long *__restrict__ kout, unsigned *__restrict__ vout, long long n, DevState *st)
{
    if (repair_keys(kin, vin, kout, vout, n, (long long)blockIdx.x * (kSortThreads * kRepairPer) + threadIdx.x))
        atomicOr(&st->status, (int)kStatLongRun);
}

// The full eight-digit sort in one co-resident kernel; does nothing unless the repair pass raised the flag.
template <int ITEMS>
__global__ void __launch_bounds__(kSortThreads, ITEMS == 16 ? 3 : 5)
sort_fallback_kernel(Workspace w, const double *__restrict__ pos, long long n, int tiles)
{
    DevState *st = w.st;
    if (!(*reinterpret_cast<volatile int *>(&st->status) & (int)kStatLongRun)) return;   // uniform over the grid
    __shared__ unsigned long long skey[(kSortThreads * ITEMS)];
    __shared__ unsigned whist[kSortThreads / 32][kRadix];
    __shared__ unsigned sbase[kRadix];
    __shared__ unsigned stmp[8];
    unsigned *bar = st->mid_bar;
    const unsigned tid = threadIdx.x;
    const long long gtid = (long long)blockIdx.x * kSortThreads + tid, gthreads = (long long)gridDim.x * kSortThreads;
    {   // the keys again (buffer 0 holds a partial result) and clean look-back rows
        const double lx = st->lo[0], ly = st->lo[1], lz = st->lo[2], sc = st->scale;
        for (long long i = gtid; i < n; i += gthreads)
            w.key[0][i] = morton_key(__ldg(pos + 3 * i), __ldg(pos + 3 * i + 1), __ldg(pos + 3 * i + 2), lx, ly, lz, sc);
        for (long long i = gtid; i < (long long)kSortPasses * tiles * kRadix; i += gthreads) w.lookback[i] = 0u;
    }
    grid_barrier(bar, gridDim.x);
    int a = 0;
    for (int p = 0; p < kSortPasses; ++p) {
        // Tiles in rounds: block b takes tiles b, b + grid, ...  All blocks are resident and a round's tiles start
        // together, so the tiles a look-back waits for are running or done.
        unsigned *lb = w.lookback + (size_t)p * tiles * kRadix;
        const int b = a ^ 1;
        for (unsigned tile = blockIdx.x; tile < (unsigned)tiles; tile += gridDim.x) {
            __syncthreads();
#pragma unroll
            for (int q = 0; q < kSortThreads / 32; ++q) whist[q][tid] = 0u;
            __syncthreads();
            const long long base = (long long)tile * (kSortThreads * ITEMS);
            const long long rem = n - base;
            const unsigned nvalid = rem >= kSortThreads * ITEMS ? (unsigned)(kSortThreads * ITEMS) : (unsigned)rem;
            if (p == 0) sort_tile<true, ITEMS, false>(w.key[a], w.idx[a], w.key[b], w.idx[b], base, nvalid, tile, 0, w.hist, lb, skey, whist, sbase, stmp);
            else sort_tile<false, ITEMS, false>(w.key[a], w.idx[a], w.key[b], w.idx[b], base, nvalid, tile, p * kRadixBits, w.hist + p * kRadix, lb, skey, whist, sbase, stmp);
        }
        a ^= 1;
        grid_barrier(bar, gridDim.x);
    }
    // the flag has done its work; it is not an error
    if (gtid == 0) atomicAnd(&st->status, ~(int)kStatLongRun);
}

// keys per tile of the streaming passes for n keys
int sort_tile_items(int64_t n) { return n < kSortSmallTileBelow ? 8 : 16; }

template <int ITEMS>
static bool launch_sort_fallback(const Workspace &w, const double *pos, int64_t n, int tiles, cudaStream_t s)
{
    static std::atomic<int> occupancy[kMaxDevices];   // resident blocks per SM + 1, per device; 0 = not asked yet
    const int dev = current_device();
    int per_sm = occupancy[dev].load(std::memory_order_relaxed) - 1;
    if (per_sm < 0) {
        if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, sort_fallback_kernel<ITEMS>, kSortThreads, 0) != cudaSuccess) per_sm = 0;
        cudaGetLastError();
        occupancy[dev].store(per_sm + 1, std::memory_order_relaxed);
    }
    if (per_sm < 1) return false;
    // test hook (tests/test_gpu_api.py): behave as if the driver refused the cooperative launch, as it may under MPS or
    // on a partition without enough free SMs
    static const bool refuse = getenv("BH_TEST_REFUSE_COOPERATIVE_SORT") != nullptr;
    if (refuse) return false;
    int blocks = per_sm * w.sms;
    if (blocks > tiles) blocks = tiles;
    Workspace wc = w;
    long long nn = n;
    void *args[] = {&wc, &pos, &nn, &tiles};
    if (cudaLaunchCooperativeKernel((const void *)sort_fallback_kernel<ITEMS>, dim3(blocks), dim3(kSortThreads), args, 0, s) != cudaSuccess) {
        cudaGetLastError();
        return false;
    }
    return true;
}

template <int ITEMS>
static void launch_sort_pass(const Workspace &w, int64_t n, int tiles, int p, int a, bool first, cudaStream_t s)
{
    const int b = a ^ 1;
    unsigned *lb = w.lookback + (size_t)p * tiles * kRadix;   // [pass][tiles of this n][256]: cleared per build
    if (first)
        sort_pass_kernel<true, ITEMS><<<tiles, kSortThreads, 0, s>>>(w.key[a], w.idx[a], w.key[b], w.idx[b], n, p * kRadixBits,
                                                                     w.hist + p * kRadix, lb, w.sort_ticket + p);
    else
        sort_pass_kernel<false, ITEMS><<<tiles, kSortThreads, 0, s>>>(w.key[a], w.idx[a], w.key[b], w.idx[b], n, p * kRadixBits,
                                                                      w.hist + p * kRadix, lb, w.sort_ticket + p);
}

// the eight plain digit passes over the full keys (key[0]/idx[0] -> ... -> key[0]/idx[0]); needs no co-resident kernel
static void launch_sort_eight(const Workspace &w, int64_t n, int items, int tiles, cudaStream_t s)
{
    for (int p = 0; p < kSortPasses; ++p) {
        if (items == 8) launch_sort_pass<8>(w, n, tiles, p, p & 1, p == 0, s);
        else launch_sort_pass<16>(w, n, tiles, p, p & 1, p == 0, s);
    }
}

// pos: the caller's positions (the fallback recomputes the keys from them)
int launch_sort(const Workspace &w, const double *pos, int64_t n, cudaStream_t s)
{
    const int items = sort_tile_items(n);
    const int tiles = (int)((n + kSortThreads * items - 1) / (kSortThreads * items));
    // the partial-key sort needs its fallback kernel, a cooperative launch: asked once per device
    static std::atomic<int> mode[kMaxDevices];   // 0 = not asked yet, 1 = partial-key sort, 2 = eight plain passes
    const int dev = current_device();
    int m = mode[dev].load(std::memory_order_relaxed);
    if (m == 0) {
        int cur = 0, coop = 0;
        cudaGetDevice(&cur);
        cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, cur);
        cudaGetLastError();
        m = coop ? 1 : 2;
        mode[dev].store(m, std::memory_order_relaxed);
    }
    if (m == 2) {
        launch_sort_eight(w, n, items, tiles, s);
        return kSortPasses;
    }
    int a = 0;
    for (int p = kHighFirst; p < kSortPasses; ++p, a ^= 1) {
        if (items == 8) launch_sort_pass<8>(w, n, tiles, p, a, p == kHighFirst, s);
        else launch_sort_pass<16>(w, n, tiles, p, a, p == kHighFirst, s);
    }
    const int rblocks = (int)((n + kSortThreads * kRepairPer - 1) / (kSortThreads * kRepairPer));
    sort_repair_kernel<<<rblocks, kSortThreads, 0, s>>>(w.key[a], w.idx[a], w.key[a ^ 1], w.idx[a ^ 1], n, w.st);
    const bool ok = items == 8 ? launch_sort_fallback<8>(w, pos, n, tiles, s) : launch_sort_fallback<16>(w, pos, n, tiles, s);
    if (ok) return (kSortPasses - kHighFirst) + 2;
    // The co-resident kernel could not be launched (the attribute said it could: MPS, a busy partition).  Without it a run of
    // more than 64 equal top key bits would stay unsorted, so this build starts its sort again with the eight plain passes
    // — histograms, tickets and look-back rows cleared, keys recomputed from the positions — and so does every later build
    // on this device.  Same permutation, bit for bit.
    mode[dev].store(2, std::memory_order_relaxed);
    const size_t zbytes = (size_t)((char *)w.lookback - (char *)w.hist) + (size_t)kSortPasses * tiles * kRadix * sizeof(unsigned);
    if (cudaMemsetAsync(w.hist, 0, zbytes, s) != cudaSuccess) return -1;      // -1: the caller reports a CUDA error
    launch_keys(w, pos, n, s);
    launch_sort_eight(w, n, items, tiles, s);
    return (kSortPasses - kHighFirst) + 1 + 1 + kSortPasses;   // five passes + repair, then keys + eight passes
}

}  // namespace bh
