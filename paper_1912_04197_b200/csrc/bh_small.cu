// bh_small.cu — steps a1-a6 for a body set that fits ONE sort tile (n <= 4096) in ONE kernel of one block.
//
// The paper's own regime is N <= 10^4 (Fig. 4), and it notes that there "the computational
// time is dominated by the octree creation".  On a B200 a build of a thousand bodies is not
// work but latency: twelve dependent launches of a few microseconds each.  Here the whole build — bounding
// cube, Morton keys, the eight radix passes, sorted bodies, octree, group boxes, monopoles — runs in one
// 1024-thread block: the keys and the permutation stay in registers and shared memory through the sort, the
// tree phases are the tile functions of the streaming kernels (bh_tree.cuh) called for each of the <= 4 tiles
// in turn, the monopoles go level by level from the deepest (no arrival counters, no fences: one
// __syncthreads per level), and the per-build clearing (child masks) is done by the block itself, so a build
// is one launch and no memset.  Every output array is the one the streaming path writes, bit for bit (same canonical
// arithmetic, same stable order), so everything downstream (walk, getters, broad phase) is unchanged.
//
// A phase reads what an earlier phase of the same block wrote to global memory: __syncthreads() orders
// that within the block, and none of those reads goes through the non-coherent path (no __ldg / const
// __restrict__ on data produced here; only the caller's pos / mass are read that way).
#include "bh_keys.cuh"
#include "bh_sort.cuh"
#include "bh_tree.cuh"

namespace bh {

constexpr int kSmallThreads = 1024;

// Eq. (2) PAPER.md:76 for node t (R21): a leaf from its bodies, an internal node from its children in ascending
// id; masses added left to right, weighted sums by fma from 0, one IEEE division; a one-body leaf copies the body.
// The same arithmetic, in the same order, as monopoles_and_records (bh_tree.cuh).
__device__ __forceinline__ double4 monopole_of(int t, const double4 *sbody, const double4 *mono, unsigned b, unsigned c,
                                               int first, unsigned kids)
{
    const double4 *src = first >= 0 ? mono + first : sbody + b;
    const unsigned cnt = first >= 0 ? kids : c;
    double4 s = src[0];
    if (first < 0 && c == 1) return s;
    double m = s.w;
    double wx = __fma_rn(s.w, s.x, 0.0), wy = __fma_rn(s.w, s.y, 0.0), wz = __fma_rn(s.w, s.z, 0.0);
    for (unsigned u = 1; u < cnt; ++u) {
        s = src[u];
        m = __dadd_rn(m, s.w);
        wx = __fma_rn(s.w, s.x, wx);
        wy = __fma_rn(s.w, s.y, wy);
        wz = __fma_rn(s.w, s.z, wz);
    }
    return make_double4(__ddiv_rn(wx, m), __ddiv_rn(wy, m), __ddiv_rn(wz, m), m);
}

template <int ITEMS>
__global__ void __launch_bounds__(kSmallThreads) build_small_kernel(Workspace w, const double *__restrict__ pos,
                                                                    const double *__restrict__ mass, int n, int C)
{
    // shared memory, reused phase by phase
    extern __shared__ __align__(16) unsigned char smem[];
    __shared__ double red[2][3][kSmallThreads / 32];
    __shared__ int redbad[kSmallThreads / 32];
    __shared__ unsigned stmp[8];
    __shared__ unsigned slv[kLevels + 2];      // level histogram / level totals / level starts, by phase
    const unsigned tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
    DevState *st = w.st;

    // ---- a1: bounding cube (R11).  min / max are exact and order-free, so any reduction shape gives the same cube
    {
        const double inf = __longlong_as_double(0x7ff0000000000000ll);
        double mn[3] = {inf, inf, inf}, mx[3] = {-inf, -inf, -inf};
        int bad = 0;
        for (int i = tid; i < n; i += kSmallThreads) {
#pragma unroll
            for (int a = 0; a < 3; ++a) {
                const double x = __ldg(pos + 3 * i + a);
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
        if (tid == 0) {
            double lo[3], hi[3];
            bad = 0;
            for (int a = 0; a < 3; ++a) {
                lo[a] = red[0][a][0];
                hi[a] = red[1][a][0];
                for (int q = 1; q < kSmallThreads / 32; ++q) {
                    lo[a] = fmin(lo[a], red[0][a][q]);
                    hi[a] = fmax(hi[a], red[1][a][q]);
                }
            }
            for (int q = 0; q < kSmallThreads / 32; ++q) bad |= redbad[q];
            finish_cube(lo, hi, bad, st);
        }
        __syncthreads();
    }

    // ---- a2 + a3: keys straight into the sort's register layout, eight passes in shared memory
    {
        unsigned long long *skey = reinterpret_cast<unsigned long long *>(smem);                  // [1024 * ITEMS]
        unsigned(*whist)[kRadix] = reinterpret_cast<unsigned(*)[kRadix]>(skey + kSmallThreads * ITEMS);   // [32][256]
        unsigned *stoff = &whist[kSmallThreads / 32][0];                                          // [256]
        const double lx = st->lo[0], ly = st->lo[1], lz = st->lo[2], sc = st->scale;
        unsigned long long k[ITEMS];
        unsigned v[ITEMS];
#pragma unroll
        for (int i = 0; i < ITEMS; ++i) {
            const int idx = warp * (32 * ITEMS) + i * 32 + lane;
            k[i] = ~0ull;
            if (idx < n) k[i] = morton_key(__ldg(pos + 3 * idx), __ldg(pos + 3 * idx + 1), __ldg(pos + 3 * idx + 2), lx, ly, lz, sc);
            v[i] = (unsigned)idx;
        }
        // the partial-key sort of bh_sort.cu inside the block: five passes over the high digits, then every key is ranked
        // within its run of equal top bits (the keys lie in shared memory for that); a run longer than kRunMax makes
        // the block sort again with all eight digits (uniform branch)
        block_radix_sort<ITEMS, kSmallThreads>(k, v, skey, whist, stoff, stmp, kHighFirst);
        int place[ITEMS];
        bool too_long = false;
#pragma unroll
        for (int i = 0; i < ITEMS; ++i) skey[warp * (32 * ITEMS) + i * 32 + lane] = k[i];     // padding keys ~0 sort last
        __syncthreads();
#pragma unroll
        for (int i = 0; i < ITEMS; ++i) {
            const int j = warp * (32 * ITEMS) + i * 32 + lane;
            place[i] = j;
            if (j >= n) continue;
            const unsigned long long top = k[i] >> kLowBits;
            int lo = j, hi = j + 1;
            while (lo > 0 && j - lo <= (int)kRunMax && (skey[lo - 1] >> kLowBits) == top) --lo;
            while (hi < n && hi - j <= (int)kRunMax && (skey[hi] >> kLowBits) == top) ++hi;
            if (hi - lo > (int)kRunMax) {
                too_long = true;
                continue;
            }
            int r = lo;
            for (int q = lo; q < hi; ++q) r += (skey[q] < k[i]) || (skey[q] == k[i] && q < j);
            place[i] = r;
        }
        if (__syncthreads_or(too_long)) {
#pragma unroll
            for (int i = 0; i < ITEMS; ++i) {
                const int idx = warp * (32 * ITEMS) + i * 32 + lane;
                k[i] = ~0ull;
                if (idx < n) k[i] = morton_key(__ldg(pos + 3 * idx), __ldg(pos + 3 * idx + 1), __ldg(pos + 3 * idx + 2), lx, ly, lz, sc);
                v[i] = (unsigned)idx;
                place[i] = idx;
            }
            block_radix_sort<ITEMS, kSmallThreads>(k, v, skey, whist, stoff, stmp);
        }
        // ---- a4: sorted keys, permutation, sorted bodies
#pragma unroll
        for (int i = 0; i < ITEMS; ++i) {
            const int j = warp * (32 * ITEMS) + i * 32 + lane;
            if (j < n) {
                const unsigned b = v[i];
                w.key[0][place[i]] = k[i];
                w.idx[0][place[i]] = b;
                w.sbody[place[i]] = make_double4(__ldg(pos + 3 * b), __ldg(pos + 3 * b + 1), __ldg(pos + 3 * b + 2), __ldg(mass + b));
            }
        }
        __syncthreads();
    }

    // ---- a5: octree from the sorted keys, tile by tile (the functions of the streaming kernels)
    const int ntiles = (n + kTreeTile - 1) / kTreeTile;
    for (int t = 0; t < ntiles; ++t) {
        tree_levels_tile(w.key[0], n, C, w.group_cell, w.group_w, w.dlev, w.tile_lvl, ntiles, t,
                         reinterpret_cast<unsigned *>(smem), slv);
        __syncthreads();
    }
    tree_scan_block(w.tile_lvl, ntiles, st, w.node_cap, w.gstart, (unsigned)n, slv);
    __syncthreads();
    const int M = st->n_nodes;
    if ((long long)M > w.node_cap) return;        // flagged; uniform over the block
    for (int t = tid; t < M; t += kSmallThreads) w.node_meta[t] = 0u;     // child masks and arrival counters
    __syncthreads();
    for (int t = 0; t < ntiles; ++t) {
        tree_emit_tile(w.key[0], n, w.dlev, w.tile_lvl, ntiles, t, st, w.node_cap, w.nlevel, w.nbegin, w.nfirst,
                       w.nparent, w.node_meta, w.gstart, reinterpret_cast<unsigned(*)[kLevels + 1]>(smem), slv);
        __syncthreads();
    }
    // ---- group boxes; a6: monopoles and the walk's node records, level by level from the deepest
    group_boxes(st->n_groups, warp, kSmallThreads / 32, w.gstart, w.sbody, w.gbox);
    if (tid <= (unsigned)kLevels) slv[tid] = st->lvl_start[tid];
    const int depth = st->depth;
    __syncthreads();
    for (int l = depth; l >= 0; --l) {
        for (int t = (int)slv[l] + (int)tid; t < (int)slv[l + 1]; t += kSmallThreads) {
            const int first = w.nfirst[t];
            const unsigned b = w.nbegin[t], c = node_count(t, M, (unsigned)n, w.nbegin, w.nparent);
            w.ncount[t] = c;
            const unsigned kids = (unsigned)__popc(__ldcg(w.node_meta + t) & 0xffu);   // masks were set by atomics (L2)
            w.winfo[t] = make_uint4(b, c, (unsigned)first, (unsigned)l | (kids << 8));
            w.mono[t] = monopole_of(t, w.sbody, w.mono, b, c, first, kids);
        }
        __syncthreads();
    }
}

template <int ITEMS>
static void launch_small_t(const Workspace &w, const double *pos, const double *mass, int n, cudaStream_t s)
{
    // sort: keys + per-warp histograms + digit offsets; tree: two window arrays / the emission's chunk counts
    size_t sort_bytes = (size_t)kSmallThreads * ITEMS * 8 + (size_t)(kSmallThreads / 32 + 1) * kRadix * 4;
    size_t tree_bytes = (size_t)tree_levels_smem_words(w.leaf_cap, w.group_cell) * sizeof(unsigned);
    size_t emit_bytes = (size_t)(kTreeTile / 32) * (kLevels + 1) * 4;
    size_t bytes = sort_bytes > tree_bytes ? sort_bytes : tree_bytes;
    if (emit_bytes > bytes) bytes = emit_bytes;
    static std::atomic<bool> configured[kMaxDevices];   // the attribute is per device
    const int dev = current_device();
    if (!configured[dev].load(std::memory_order_relaxed)) {
        cudaFuncSetAttribute(build_small_kernel<ITEMS>, cudaFuncAttributeMaxDynamicSharedMemorySize, 96 * 1024);
        configured[dev].store(true, std::memory_order_relaxed);
    }
    build_small_kernel<ITEMS><<<1, kSmallThreads, bytes, s>>>(w, pos, mass, n, w.leaf_cap);
}

// n <= kSortTile (4096)
void launch_build_small(const Workspace &w, const double *pos, const double *mass, int64_t n, cudaStream_t s)
{
    if (n <= kSmallThreads) launch_small_t<1>(w, pos, mass, (int)n, s);
    else if (n <= kSmallThreads * 2) launch_small_t<2>(w, pos, mass, (int)n, s);
    else launch_small_t<4>(w, pos, mass, (int)n, s);
}

}  // namespace bh
