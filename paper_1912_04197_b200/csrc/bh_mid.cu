// bh_mid.cu — steps a1-a6 for a mid-size body set (one sort tile < n <= one tree tile per SM) in ONE kernel.
//
// Between the one-block build (n <= 4096, bh_small.cu) and the sizes where the streaming kernels are bound by
// work, a build is bound by its sixteen dependent launches (and two memsets): a kernel of a few thousand bodies per SM ends a few
// microseconds after it starts, and the next one cannot start before (N = 16 384: 135 us for ~15 us of work; the
// paper's own regime is N <= 10^4 .. 10^5).  Here the same phases — cube, keys + histograms,
// the digit passes and the repair of the partial-key sort, gather, tree levels / scan / emission, group boxes, monopoles — run in one co-resident grid
// (at most one 256-thread block per SM, cooperative launch) with a grid barrier where a launch boundary was.
// Every phase is the tile / block function of the streaming kernels (bh_sort.cuh, bh_tree.cuh, bh_keys.cuh), so every
// output array is the streaming path's, bit for bit.
//
// Coherence.  A phase reads what OTHER blocks wrote in an earlier phase of the same kernel (the sort's ping-pong
// buffers are read, rewritten by other SMs and read again).  The barrier between phases orders the accesses and drops
// the L1: the grid barrier arrives with an acq_rel atomic and waits with ld.acquire.gpu (LDG.STRONG.GPU + CCTL.IVALL on
// sm_100, bh_grid.cuh), the cluster barrier is MEMBAR.ALL.GPU / UCGABAR / CCTL.IVALL — so the plain loads of the next
// phase cannot hit a stale line (what cooperative-groups grid.sync() rests on as well).  No pointer to data produced
// here is const __restrict__ / __ldg (only the caller's pos / mass are read that way).
#include "bh_keys.cuh"
#include "bh_sort.cuh"
#include "bh_tree.cuh"
#include "bh_grid.cuh"

namespace bh {

constexpr int kMidThreads = kSortThreads;   // 256: the sort tile's block size
constexpr int kMidItems = 8;                // 2048-key sort tiles, as the streaming passes below kSortSmallTileBelow keys (1024- and 512-key
                                            // tiles change a pass by < 0.5 us: a pass is 3 us of tile chain + 2.3 us of barrier)

// One thread-block CLUSTER (the whole grid: 8 blocks): the hardware barrier of the cluster.  Its arrive has release,
// its wait acquire semantics (SASS: MEMBAR.ALL.GPU, UCGABAR_ARV / UCGABAR_WAIT, CCTL.IVALL), so it orders global memory
// between the blocks and drops the L1 like the grid barrier does, without a round trip through an atomic in the L2.
__device__ __forceinline__ void cluster_barrier()
{
    asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory");
    asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory");
}

template <bool CLUSTER>
__device__ __forceinline__ void phase_barrier(unsigned *bar)
{
    if constexpr (CLUSTER) cluster_barrier();
    else grid_barrier(bar, gridDim.x);
}

template <bool CLUSTER>
__global__ void __launch_bounds__(kMidThreads) build_mid_kernel(Workspace w, const double *__restrict__ pos,
                                                                const double *__restrict__ mass, int n, int C,
                                                                int sort_tiles, int tree_tiles, long long node_words)
{
    extern __shared__ __align__(16) unsigned char smem[];
    __shared__ double red[2][3][kMidThreads / 32];
    __shared__ int redbad[kMidThreads / 32];
    __shared__ unsigned stmp[8];
    __shared__ unsigned slv[kLevels + 2];
    const unsigned tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
    const int gtid = blockIdx.x * kMidThreads + (int)tid, gthreads = gridDim.x * kMidThreads;
    DevState *st = w.st;
    unsigned *bar = st->mid_bar;

    // ---- what a streaming build clears with two memsets: histograms, look-back rows of this n, child masks / counters
    for (int k = gtid; k < kSortPasses * kRadix; k += gthreads) w.hist[k] = 0u;
    for (long long k = gtid; k < (long long)kSortPasses * sort_tiles * kRadix; k += gthreads) w.lookback[k] = 0u;
    for (long long k = gtid; k < node_words; k += gthreads) w.node_meta[k] = 0u;

    // ---- a1: bounding cube (R11): per-block extremes, then block 0 derives the cube (min / max are exact and order-free)
    {
        const double inf = __longlong_as_double(0x7ff0000000000000ll);
        double mn[3] = {inf, inf, inf}, mx[3] = {-inf, -inf, -inf};
        int bad = 0;
        for (int i = gtid; i < n; i += gthreads) {
#pragma unroll
            for (int a = 0; a < 3; ++a) {
                const double x = __ldg(pos + 3 * (long long)i + a);
                bad |= nonfinite(x);
                mn[a] = fmin(mn[a], x);
                mx[a] = fmax(mx[a], x);
            }
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
#pragma unroll
            for (int a = 0; a < 3; ++a) {
                mn[a] = fmin(mn[a], __shfl_xor_sync(0xffffffffu, mn[a], o));
                mx[a] = fmax(mx[a], __shfl_xor_sync(0xffffffffu, mx[a], o));
            }
            bad |= __shfl_xor_sync(0xffffffffu, bad, o);
        }
        if (lane == 0) {
#pragma unroll
            for (int a = 0; a < 3; ++a) {
                red[0][a][warp] = mn[a];
                red[1][a][warp] = mx[a];
            }
            redbad[warp] = bad;
        }
        __syncthreads();
        if (tid < 3) {
            double lo = red[0][tid][0], hi = red[1][tid][0];
            for (int q = 1; q < kMidThreads / 32; ++q) {
                lo = fmin(lo, red[0][tid][q]);
                hi = fmax(hi, red[1][tid][q]);
            }
            w.bbox_part[blockIdx.x * 8 + tid] = lo;
            w.bbox_part[blockIdx.x * 8 + 3 + tid] = hi;
        }
        if (tid == 0) {
            int b = 0;
            for (int q = 0; q < kMidThreads / 32; ++q) b |= redbad[q];
            w.bbox_part[blockIdx.x * 8 + 6] = b ? 1.0 : 0.0;
        }
        phase_barrier<CLUSTER>(bar);
        if (blockIdx.x == 0 && warp == 0) {       // one warp: lanes take the blocks' rows in turn, then a shuffle reduction
            double lo[3] = {inf, inf, inf}, hi[3] = {-inf, -inf, -inf};
            int b = 0;
            for (unsigned q = lane; q < gridDim.x; q += 32) {
#pragma unroll
                for (int a = 0; a < 3; ++a) {
                    lo[a] = fmin(lo[a], w.bbox_part[q * 8 + a]);
                    hi[a] = fmax(hi[a], w.bbox_part[q * 8 + 3 + a]);
                }
                b |= (w.bbox_part[q * 8 + 6] != 0.0);
            }
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
#pragma unroll
                for (int a = 0; a < 3; ++a) {
                    lo[a] = fmin(lo[a], __shfl_xor_sync(0xffffffffu, lo[a], o));
                    hi[a] = fmax(hi[a], __shfl_xor_sync(0xffffffffu, hi[a], o));
                }
                b |= __shfl_xor_sync(0xffffffffu, b, o);
            }
            if (lane == 0) finish_cube(lo, hi, b, st);
        }
        phase_barrier<CLUSTER>(bar);
    }

    // ---- a2: keys + the eight digit histograms
    {
        unsigned *sh = reinterpret_cast<unsigned *>(smem);   // [8][256]
        for (int k = tid; k < kSortPasses * kRadix; k += kMidThreads) sh[k] = 0u;
        __syncthreads();
        const double lx = st->lo[0], ly = st->lo[1], lz = st->lo[2], sc = st->scale;
        for (int i = gtid; i < n; i += gthreads) {
            const unsigned long long k = morton_key(__ldg(pos + 3 * (long long)i), __ldg(pos + 3 * (long long)i + 1),
                                                    __ldg(pos + 3 * (long long)i + 2), lx, ly, lz, sc);
            w.key[0][i] = k;
#pragma unroll
            for (int p = 0; p < kSortPasses; ++p)
                atomicAdd(&sh[p * kRadix + (unsigned)((k >> (p * kRadixBits)) & (kRadix - 1))], 1u);
        }
        __syncthreads();
        for (int k = tid; k < kSortPasses * kRadix; k += kMidThreads)
            if (sh[k]) atomicAdd(&w.hist[k], sh[k]);
        phase_barrier<CLUSTER>(bar);
    }

    // ---- a3: the sort, as above 1024 bodies per SM (bh_sort.cu): digit passes over the five high digits, a repair pass that
    //      orders the runs of equal top bits, and — a uniform branch here, not a kernel — all eight digits from scratch if
    //      a run was too long.  Block b sorts tiles b, b + grid, ... in ascending order (the look-back of a tile only waits
    //      for lower tiles, and every block is resident).
    {
        unsigned long long *skey = reinterpret_cast<unsigned long long *>(smem);                          // [256 * 8]
        unsigned(*whist)[kRadix] = reinterpret_cast<unsigned(*)[kRadix]>(skey + kMidThreads * kMidItems);   // [8][256]
        unsigned *sbase = &whist[kMidThreads / 32][0];                                                    // [256]
        const unsigned sorters = (unsigned)sort_tiles < gridDim.x ? (unsigned)sort_tiles : gridDim.x;   // blocks that own tiles
        // digits p0 .. 7 starting from buffer 0 (values = positions in the first of them)
        auto digit_passes = [&](int p0) {
            int a = 0;
            for (int p = p0; p < kSortPasses && (CLUSTER || blockIdx.x < sorters); ++p, a ^= 1) {
                const int b = a ^ 1;
                unsigned *lb = w.lookback + (size_t)p * sort_tiles * kRadix;
                for (int tile = blockIdx.x; tile < sort_tiles; tile += gridDim.x) {
#pragma unroll
                    for (int q = 0; q < kMidThreads / 32; ++q) whist[q][tid] = 0u;
                    __syncthreads();
                    const long long base = (long long)tile * (kMidThreads * kMidItems);
                    const long long rem = n - base;
                    const unsigned nvalid = rem >= kMidThreads * kMidItems ? (unsigned)(kMidThreads * kMidItems) : (unsigned)rem;
                    if (p == p0) sort_tile<true, kMidItems, false>(w.key[a], w.idx[a], w.key[b], w.idx[b], base, nvalid, tile, p * kRadixBits, w.hist + p * kRadix, lb, skey, whist, sbase, stmp);
                    else sort_tile<false, kMidItems, false>(w.key[a], w.idx[a], w.key[b], w.idx[b], base, nvalid, tile, p * kRadixBits, w.hist + p * kRadix, lb, skey, whist, sbase, stmp);
                    __syncthreads();
                }
                if (p + 1 < kSortPasses) {     // between passes: the whole cluster, or the sorting blocks of the grid only
                    if constexpr (CLUSTER) cluster_barrier();
                    else grid_barrier(bar + 2, sorters);
                }
            }
            phase_barrier<CLUSTER>(bar);       // after the last pass: everybody
        };
        digit_passes(kHighFirst);              // five passes: the result is in buffer 1
        bool too_long = false;
        for (long long j0 = (long long)blockIdx.x * (kMidThreads * kRepairPer) + tid; j0 < n; j0 += (long long)gridDim.x * (kMidThreads * kRepairPer))
            too_long |= repair_keys(w.key[1], w.idx[1], w.key[0], w.idx[0], n, j0);
        if (too_long) atomicOr(&st->status, (int)kStatLongRun);
        phase_barrier<CLUSTER>(bar);
        if (*reinterpret_cast<volatile int *>(&st->status) & (int)kStatLongRun) {   // uniform over the grid
            const double lx = st->lo[0], ly = st->lo[1], lz = st->lo[2], sc = st->scale;
            for (int i = gtid; i < n; i += gthreads)
                w.key[0][i] = morton_key(__ldg(pos + 3 * (long long)i), __ldg(pos + 3 * (long long)i + 1),
                                         __ldg(pos + 3 * (long long)i + 2), lx, ly, lz, sc);
            for (long long k = gtid; k < (long long)kSortPasses * sort_tiles * kRadix; k += gthreads) w.lookback[k] = 0u;
            phase_barrier<CLUSTER>(bar);
            digit_passes(0);                   // eight passes: the result is in buffer 0
            if (gtid == 0) atomicAnd(&st->status, ~(int)kStatLongRun);   // the flag has done its work; it is not an error
        }
    }

    // ---- a4: sorted bodies
    for (int j = gtid; j < n; j += gthreads) {
        const unsigned i = w.idx[0][j];
        w.sbody[j] = make_double4(__ldg(pos + 3ll * i), __ldg(pos + 3ll * i + 1), __ldg(pos + 3ll * i + 2), __ldg(mass + i));
    }
    // (the tree phases read the keys only; the sorted bodies are first read after the barriers below)

    // ---- a5: octree from the sorted keys
    for (int t = blockIdx.x; t < tree_tiles; t += gridDim.x) {
        tree_levels_tile(w.key[0], n, C, w.group_cell, w.group_w, w.dlev, w.tile_lvl, tree_tiles, t,
                         reinterpret_cast<unsigned *>(smem), slv);
        __syncthreads();
    }
    phase_barrier<CLUSTER>(bar);
    if (blockIdx.x == 0) tree_scan_block(w.tile_lvl, tree_tiles, st, w.node_cap, w.gstart, (unsigned)n, slv);
    phase_barrier<CLUSTER>(bar);
    const int M = st->n_nodes;
    if ((long long)M > w.node_cap) return;        // flagged by the scan; uniform over the grid
    for (int t = blockIdx.x; t < tree_tiles; t += gridDim.x) {
        tree_emit_tile(w.key[0], n, w.dlev, w.tile_lvl, tree_tiles, t, st, w.node_cap, w.nlevel, w.nbegin, w.nfirst,
                       w.nparent, w.node_meta, w.gstart, reinterpret_cast<unsigned(*)[kLevels + 1]>(smem), slv);
        __syncthreads();
    }
    phase_barrier<CLUSTER>(bar);

    // ---- group boxes; a6: monopoles, node counts and the walk's node records (arrival counters, as monopole_kernel)
    group_boxes(st->n_groups, (unsigned)(gtid >> 5), (unsigned)(gthreads >> 5), w.gstart, w.sbody, w.gbox);
    monopoles_and_records(M, (unsigned)n, gtid, gthreads, w.sbody, w.nbegin, w.ncount, w.nfirst, w.nparent, w.node_meta,
                          w.mono, w.nlevel, w.winfo);
}

// largest n the one-kernel build takes: one tree tile per SM (so every block has at most one tile per phase)
int64_t mid_build_limit(const Workspace &w) { return (int64_t)w.sms * kTreeTile; }

int launch_build_mid(const Workspace &w, const double *pos, const double *mass, int64_t n, cudaStream_t s)
{
    const int sort_tiles = (int)((n + kMidThreads * kMidItems - 1) / (kMidThreads * kMidItems));
    const int tree_tiles = (int)((n + kTreeTile - 1) / kTreeTile);
    int blocks = w.sms;    // every SM: the streaming phases (cube, keys, gather, boxes, monopoles) use them all
    size_t sort_bytes = (size_t)kMidThreads * kMidItems * 8 + (size_t)(kMidThreads / 32 + 1) * kRadix * 4;
    size_t tree_bytes = (size_t)tree_levels_smem_words(w.leaf_cap, w.group_cell) * sizeof(unsigned);
    size_t emit_bytes = (size_t)(kTreeTile / 32) * (kLevels + 1) * 4;
    size_t hist_bytes = (size_t)kSortPasses * kRadix * 4;
    size_t bytes = sort_bytes > tree_bytes ? sort_bytes : tree_bytes;
    if (emit_bytes > bytes) bytes = emit_bytes;
    if (hist_bytes > bytes) bytes = hist_bytes;
    int nn = (int)n, C = w.leaf_cap, st_ = sort_tiles, tt = tree_tiles;
    long long node_words = node_capacity(n, w.leaf_cap);
    Workspace wc = w;
    void *args[] = {&wc, &pos, &mass, &nn, &C, &st_, &tt, &node_words};
    // At most one tree tile per block of ONE portable cluster (8 blocks, n <= 8192): the cluster's hardware barrier (a step
    // at N = 4200 .. 8000 is 11 - 15 us shorter than with the grid barrier; with two tiles per block it is 25 us longer).
    if (tree_tiles <= 8) {
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3(8);
        cfg.blockDim = dim3(kMidThreads);
        cfg.dynamicSmemBytes = bytes;
        cfg.stream = s;
        cudaLaunchAttribute at[1];
        at[0].id = cudaLaunchAttributeClusterDimension;
        at[0].val.clusterDim.x = 8;
        at[0].val.clusterDim.y = 1;
        at[0].val.clusterDim.z = 1;
        cfg.attrs = at;
        cfg.numAttrs = 1;
        cudaError_t ec = cudaLaunchKernelEx(&cfg, build_mid_kernel<true>, wc, pos, mass, nn, C, st_, tt, node_words);
        if (ec == cudaSuccess) return 1;
        cudaGetLastError();            // fall through to the grid version
    }
    // cooperative: the runtime guarantees that all blocks are resident together (a plain launch costs the same here)
    cudaError_t e = cudaLaunchCooperativeKernel((const void *)build_mid_kernel<false>, dim3(blocks), dim3(kMidThreads), args, bytes, s);
    return e == cudaSuccess ? 1 : -1;
}

}  // namespace bh
