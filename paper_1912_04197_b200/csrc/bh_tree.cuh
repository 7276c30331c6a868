// bh_tree.cuh — block-level bodies of steps a4-a6 (group boxes, octree from the sorted keys, monopoles), shared by
// the streaming kernels of bh_tree.cu (one call per thread block) and the one-block build of small body sets
// (bh_small.cu: the same functions called for every tile in turn).  See bh_tree.cu for the derivation.
// Pointers to data that the build itself produces are NOT const __restrict__ here: in the one-block build a phase
// reads what an earlier phase of the same kernel wrote, which must not go through the non-coherent load path.
#pragma once
#include "bh_common.cuh"

namespace bh {

// Order-preserving map of a finite double onto an unsigned 64-bit integer (and back): min / max of doubles become
// integer min / max, which the warp computes with two REDUX instructions per quantity (high words, then the low
// words of the lanes that tie on the high word) instead of five rounds of 64-bit shuffles and fp64 min / max.
__device__ __forceinline__ unsigned long long ordered_bits(double x)
{
    const unsigned long long u = (unsigned long long)__double_as_longlong(x);
    return (u >> 63) ? ~u : (u | 0x8000000000000000ull);
}
__device__ __forceinline__ double from_ordered_bits(unsigned long long k)
{
    const unsigned long long u = (k >> 63) ? (k & 0x7fffffffffffffffull) : ~k;
    return __longlong_as_double((long long)u);
}
__device__ __forceinline__ unsigned long long warp_min_u64(unsigned long long k)
{
    const unsigned hi = (unsigned)(k >> 32);
    const unsigned mh = __reduce_min_sync(0xffffffffu, hi);
    const unsigned ml = __reduce_min_sync(0xffffffffu, hi == mh ? (unsigned)k : 0xffffffffu);
    return ((unsigned long long)mh << 32) | ml;
}
__device__ __forceinline__ unsigned long long warp_max_u64(unsigned long long k)
{
    const unsigned hi = (unsigned)(k >> 32);
    const unsigned mh = __reduce_max_sync(0xffffffffu, hi);
    const unsigned ml = __reduce_max_sync(0xffffffffu, hi == mh ? (unsigned)k : 0u);
    return ((unsigned long long)mh << 32) | ml;
}

// exact bounding box of every walk group: warp `wid` of `nwarps` takes groups wid, wid + nwarps, ...
__device__ __forceinline__ void group_boxes(unsigned ng, unsigned wid, unsigned nwarps, const unsigned *gstart,
                                            const double4 *sbody, double *gbox)
{
    const unsigned lane = lane_id();
    for (unsigned g = wid; g < ng; g += nwarps) {
        const unsigned b = gstart[g], e = gstart[g + 1];
        // every lane starts from the group's first body, so lanes beyond a short group are neutral
        double4 p = sbody[b + lane < e ? b + lane : b];
        double lx = p.x, ly = p.y, lz = p.z, hx = p.x, hy = p.y, hz = p.z;
        for (unsigned j = b + lane + 32; j < e; j += 32) {      // W <= 32: at most one body per lane; kept general
            p = sbody[j];
            lx = fmin(lx, p.x); ly = fmin(ly, p.y); lz = fmin(lz, p.z);
            hx = fmax(hx, p.x); hy = fmax(hy, p.y); hz = fmax(hz, p.z);
        }
        const unsigned long long rlx = warp_min_u64(ordered_bits(lx)), rly = warp_min_u64(ordered_bits(ly)),
                                 rlz = warp_min_u64(ordered_bits(lz)), rhx = warp_max_u64(ordered_bits(hx)),
                                 rhy = warp_max_u64(ordered_bits(hy)), rhz = warp_max_u64(ordered_bits(hz));
        if (lane == 0) {
            double *q = gbox + 6ull * g;
            q[0] = from_ordered_bits(rlx); q[1] = from_ordered_bits(rly); q[2] = from_ordered_bits(rlz);
            q[3] = from_ordered_bits(rhx); q[4] = from_ordered_bits(rhy); q[5] = from_ordered_bits(rhz);
        }
    }
}

// Sliding maximum over windows of k consecutive entries of a signed-byte array of nw 32-bit words (entries past
// the data are -1, the neutral value), four entries per operation: after r rounds x[i] = max(x[i .. i + 2^r - 1]).
// Runs p = floor(log2 k) rounds, ping-ponging between a and b; *out is the array that holds the result, and the
// caller combines out[i] and out[i + k - 2^p].  Returns 2^p.
__device__ __forceinline__ int window_doubling(unsigned *a, unsigned *b, int nw, int k, const signed char **out)
{
    int p = 0;
    while ((2 << p) <= k) ++p;
    for (int r = 0; r < p; ++r) {
        const int h = 1 << r;                 // entries (bytes) to look ahead
        for (int i = threadIdx.x; i < nw; i += blockDim.x) {
            const unsigned x = a[i];
            unsigned y;
            if (h >= 4) {
                const int j = i + (h >> 2);
                y = j < nw ? a[j] : 0xffffffffu;
            } else {
                const unsigned nxt = i + 1 < nw ? a[i + 1] : 0xffffffffu;
                y = __funnelshift_r(x, nxt, 8 * h);     // entries 4 i + h .. 4 i + h + 3 (little endian)
            }
            b[i] = __vmaxs4(x, y);
        }
        __syncthreads();
        unsigned *t = a; a = b; b = t;
    }
    *out = reinterpret_cast<const signed char *>(a);
    return 1 << p;
}

// first index <= j whose key shares its leading `lvl` digits with key j (galloping search)
__device__ __forceinline__ unsigned range_begin(const unsigned long long *skey, unsigned j, int lvl)
{
    if (lvl == 0) return 0u;
    const int sh = 63 - 3 * lvl;
    const unsigned long long pre = skey[j] >> sh;
    unsigned hi = j, step = 1, lo;          // invariant: key[hi] has the prefix
    while (true) {
        if (hi < step) { lo = 0u; if ((skey[0] >> sh) == pre) return 0u; break; }
        lo = hi - step;
        if ((skey[lo] >> sh) != pre) break;
        hi = lo;
        step <<= 1;
    }
    // key[lo] lacks the prefix, key[hi] has it: answer in (lo, hi]
    while (hi - lo > 1) {
        unsigned mid = lo + ((hi - lo) >> 1);
        if ((skey[mid] >> sh) == pre) hi = mid; else lo = mid;
    }
    return hi;
}

// first index > j (<= n) whose key differs from key j in its leading `lvl` digits (galloping search)
__device__ __forceinline__ unsigned range_end(const unsigned long long *skey, unsigned n, unsigned j, int lvl)
{
    if (lvl == 0) return n;
    const int sh = 63 - 3 * lvl;
    const unsigned long long pre = skey[j] >> sh;
    unsigned lo = j, step = 1;               // invariant: key[lo] has the prefix
    unsigned hi;
    while (true) {
        hi = lo + step;
        if (hi >= n) { hi = n; break; }
        if ((skey[hi] >> sh) != pre) break;
        lo = hi;
        step <<= 1;
    }
    // answer in (lo, hi]
    while (hi - lo > 1) {
        unsigned mid = lo + ((hi - lo) >> 1);
        if ((skey[mid] >> sh) == pre) lo = mid; else hi = mid;
    }
    return hi;
}

// words of shared memory tree_levels_tile needs for leaf capacity C and group-cell capacity Gc
__host__ __device__ inline int tree_levels_smem_words(int C, int Gc)
{
    return 2 * ((kTreeTile + C + 3) / 4) + 2 * ((kTreeTile + Gc + 3) / 4) + kTreeTile + 64;
}

// Tile `tile` of kTreeTile bodies, any block size >= 256: per body (d+1, leaf, group-start flag, group-cell level)
// and the tile's counts of nodes per level and of group starts.  sw: tree_levels_smem_words(C, Gc) words of shared
// memory; shist: kLevels + 1 words.
__device__ __forceinline__ void tree_levels_tile(const unsigned long long *skey, long long n, int C, int Gc, int W,
                                                 uchar4 *dlev, unsigned *tile_lvl, int ntiles, int tile,
                                                 unsigned *sw, unsigned *shist)
{
    const int nwc = (kTreeTile + C + 3) / 4, nwg = (kTreeTile + Gc + 3) / 4;
    unsigned *wc0 = sw, *wc1 = wc0 + nwc, *wg0 = wc1 + nwc, *wg1 = wg0 + nwg;
    int *cellpos = reinterpret_cast<int *>(wg1 + nwg);          // [kTreeTile] then [32] chunk maxima, [1] tile's cell begin
    int *chunkmax = cellpos + kTreeTile;
    signed char *bc = reinterpret_cast<signed char *>(wc0), *bg = reinterpret_cast<signed char *>(wg0);
    const long long t0 = (long long)tile * kTreeTile;
    const unsigned lane = lane_id(), warp = threadIdx.x >> 5;
    const int nwarps = blockDim.x >> 5;
    if (threadIdx.x <= kLevels) shist[threadIdx.x] = 0u;
    for (int k = threadIdx.x; k < 4 * nwc; k += blockDim.x) {
        long long s = t0 - C + k;
        int wv = -1;
        if (k < kTreeTile + C && s >= 0 && s + C < n) wv = common_levels(skey[s], skey[s + C]);
        bc[k] = (signed char)wv;
    }
    for (int k = threadIdx.x; k < 4 * nwg; k += blockDim.x) {
        long long s = t0 - Gc + k;
        int wv = -1;
        if (k < kTreeTile + Gc && s >= 0 && s + Gc < n) wv = common_levels(skey[s], skey[s + Gc]);
        bg[k] = (signed char)wv;
    }
    __syncthreads();
    const signed char *swc, *swg;
    const int pc = window_doubling(wc0, wc1, nwc, C + 1, &swc);
    const int pg = window_doubling(wg0, wg1, nwg, Gc + 1, &swg);
    // per body: levels, and where its group cell begins.  Body s is the first of its group cell iff it shares fewer
    // than glev_s digits with its predecessor (d_s < glev_s); the cell of body j begins at the last such s <= j:
    // an inclusive maximum scan of (first ? s : -1) over the tile.  Bodies before the tile's first cell start
    // belong to the cell of the tile's first body, whose beginning one thread finds by search.
    for (int c = warp; c < kTreeTile / 32; c += nwarps) {
        const int k = c * 32 + (int)lane;
        const long long j = t0 + k;
        int d = -1, leaf = 0, glev = 0, mark = -1;
        if (j < n) {
            // windows of C+1 (Gc+1) bodies that start at j-C .. j  (j-Gc .. j)
            const int mw = max((int)swc[k], (int)swc[k + C + 1 - pc]);
            const int mg = max((int)swg[k], (int)swg[k + Gc + 1 - pg]);
            leaf = min(kMaxLevel, mw + 1);
            glev = min(leaf, mg + 1);
            d = (j == 0) ? -1 : common_levels(skey[j - 1], skey[j]);
            if (d < glev) mark = k;
            if (k == 0) chunkmax[32] = (int)range_begin(skey, (unsigned)j, glev);
        }
        int run = mark;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int t = __shfl_up_sync(0xffffffffu, run, o);
            if (lane >= (unsigned)o) run = max(run, t);
        }
        cellpos[k] = run;
        if (lane == 31) chunkmax[c] = run;
        // level histogram: one ballot per level that occurs in this chunk
        const int lo = __reduce_min_sync(0xffffffffu, j < n ? d + 1 : kLevels), hi = __reduce_max_sync(0xffffffffu, j < n ? leaf : -1);
        for (int l = lo; l <= hi; ++l) {
            const unsigned m = __ballot_sync(0xffffffffu, j < n && d + 1 <= l && l <= leaf);
            if (lane == 0 && m) atomicAdd(&shist[l], (unsigned)__popc(m));
        }
        // keep (d + 1, leaf, glev) for the second pass in the output array itself
        if (j < n) dlev[j] = make_uchar4((unsigned char)(d + 1), (unsigned char)leaf, 0, (unsigned char)glev);
    }
    __syncthreads();
    for (int c = warp; c < kTreeTile / 32; c += nwarps) {
        const int k = c * 32 + (int)lane;
        const long long j = t0 + k;
        int before = -1;                                   // last cell start in the chunks before this one
        for (int q = (int)lane; q < c; q += 32) before = max(before, chunkmax[q]);
        before = __reduce_max_sync(0xffffffffu, before);
        bool gs = false;
        if (j < n) {
            const int at = max(cellpos[k], before);
            const unsigned cb = at >= 0 ? (unsigned)(t0 + at) : (unsigned)chunkmax[32];
            gs = (((unsigned)j - cb) % (unsigned)W) == 0u;
            if (gs) reinterpret_cast<unsigned char *>(dlev + j)[2] = 1;
        }
        const unsigned m = __ballot_sync(0xffffffffu, gs);
        if (lane == 0 && m) atomicAdd(&shist[kLevels], (unsigned)__popc(m));
    }
    __syncthreads();
    if (threadIdx.x <= kLevels) tile_lvl[(size_t)threadIdx.x * ntiles + tile] = shist[threadIdx.x];
}

// One block: exclusive scan of the tile counts of each level (a warp per level, warps striding over the levels),
// level starts, node count, depth, group count.  stot: kLevels + 1 words of shared memory.
__device__ __forceinline__ void tree_scan_block(unsigned *tile_lvl, int ntiles, DevState *st, long long node_cap,
                                                unsigned *gstart, unsigned n, unsigned *stot)
{
    const unsigned lane = lane_id();
    const int nwarps = blockDim.x >> 5;
    for (int l = threadIdx.x >> 5; l <= kLevels; l += nwarps) {
        unsigned *row = tile_lvl + (size_t)l * ntiles;
        unsigned run = 0;
        for (int b = 0; b < ntiles; b += 32) {
            int t = b + lane;
            unsigned v = t < ntiles ? row[t] : 0u;
            unsigned inc = v;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                unsigned u = __shfl_up_sync(0xffffffffu, inc, o);
                if (lane >= (unsigned)o) inc += u;
            }
            if (t < ntiles) row[t] = run + inc - v;
            run += __shfl_sync(0xffffffffu, inc, 31);
        }
        if (lane == 0) stot[l] = run;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        unsigned acc = 0;
        int depth = 0;
        for (int k = 0; k < kLevels; ++k) {
            st->lvl_start[k] = acc;
            acc += stot[k];
            if (stot[k]) depth = k;
        }
        st->lvl_start[kLevels] = acc;
        st->n_nodes = (int)acc;
        st->depth = depth;
        st->n_groups = stot[kLevels];
        gstart[stot[kLevels]] = n;
        if ((long long)acc > node_cap) atomicOr(&st->status, (int)kStatCapacity);
    }
}

// Tile `tile`, any block size: emit the nodes.  One warp handles 32 consecutive bodies at a time; for each level a
// ballot gives the rank of the bodies that start a node there.  scnt: [kTreeTile / 32][kLevels + 1] words of
// shared memory, sstart: kLevels + 1 words.
__device__ __forceinline__ void tree_emit_tile(const unsigned long long *skey, long long n, const uchar4 *dlev,
                                               const unsigned *tile_lvl, int ntiles, int tile, const DevState *st,
                                               long long node_cap, unsigned char *nlevel, unsigned *nbegin,
                                               int *nfirst, int *nparent, unsigned *node_meta,
                                               unsigned *gstart, unsigned (*scnt)[kLevels + 1], unsigned *sstart)
{
    constexpr int kChunks = kTreeTile / 32;          // 32 chunks of 32 bodies
    const unsigned lane = lane_id(), warp = threadIdx.x >> 5;
    const int nwarps = blockDim.x >> 5;
    const long long t0 = (long long)tile * kTreeTile;
    if (threadIdx.x <= kLevels) sstart[threadIdx.x] = st->lvl_start[threadIdx.x];
    if ((long long)st->n_nodes > node_cap) return;   // flagged by the scan; stay in bounds (uniform over the block)
    // phase 1: per chunk level counts
    // (only the levels that occur in a chunk of 32 sorted bodies are visited: a handful of the 22)
    for (int c = warp; c < kChunks; c += nwarps) {
        long long j = t0 + c * 32 + lane;
        uchar4 dl = j < n ? dlev[j] : make_uchar4(255, 0, 0, 0);
        if (lane < (unsigned)kLevels) scnt[c][lane] = 0u;
        __syncwarp();
        const int lo = __reduce_min_sync(0xffffffffu, (int)dl.x), hi = __reduce_max_sync(0xffffffffu, j < n ? (int)dl.y : -1);
        for (int l = lo; l <= hi; ++l) {
            unsigned b = __ballot_sync(0xffffffffu, (int)dl.x <= l && l <= (int)dl.y);
            if (lane == 0) scnt[c][l] = __popc(b);
        }
        unsigned bg = __ballot_sync(0xffffffffu, dl.z != 0);
        if (lane == 0) scnt[c][kLevels] = __popc(bg);
    }
    __syncthreads();
    if (threadIdx.x <= kLevels) {
        unsigned run = tile_lvl[(size_t)threadIdx.x * ntiles + tile];
        for (int c = 0; c < kChunks; ++c) {
            unsigned v = scnt[c][threadIdx.x];
            scnt[c][threadIdx.x] = run;
            run += v;
        }
    }
    __syncthreads();
    // phase 2: ids and emission
    const unsigned le = (lane == 31) ? 0xffffffffu : ((2u << lane) - 1u);
    for (int c = warp; c < kChunks; c += nwarps) {
        long long j = t0 + c * 32 + lane;
        uchar4 dl = j < n ? dlev[j] : make_uchar4(255, 0, 0, 0);
        const int first = dl.x, leaf = dl.y;
        {   // group starts, numbered in sorted-body order
            const unsigned bg = __ballot_sync(0xffffffffu, dl.z != 0);
            if (dl.z) gstart[scnt[c][kLevels] + __popc(bg & le) - 1u] = (unsigned)j;
        }
        // inclusive per-level counts at this body: prev (l-1), cur (l), next (l+1); levels lo .. hi of this chunk
        const int lo = __reduce_min_sync(0xffffffffu, first), hi = __reduce_max_sync(0xffffffffu, j < n ? leaf : -1);
        unsigned pprev = 0, pcur = 0, pnext;
        if (lo <= hi) {
            if (lo > 0) {
                unsigned b = __ballot_sync(0xffffffffu, first <= lo - 1 && lo - 1 <= leaf);   // none starts there; bodies inside count
                pprev = scnt[c][lo - 1] + __popc(b & le);
            }
            unsigned b = __ballot_sync(0xffffffffu, first <= lo && lo <= leaf);
            pcur = scnt[c][lo] + __popc(b & le);
        }
#pragma unroll 1
        for (int l = lo; l <= hi; ++l) {
            pnext = 0;
            if (l + 1 < kLevels) {
                unsigned b = __ballot_sync(0xffffffffu, first <= l + 1 && l + 1 <= leaf);
                pnext = scnt[c][l + 1] + __popc(b & le);
            }
            if (first <= l && l <= leaf) {
                const unsigned id = sstart[l] + pcur - 1u;
                const int par = l ? (int)(sstart[l - 1] + pprev - 1u) : -1;
                const bool internal = l < leaf;
                nlevel[id] = (unsigned char)l;
                nbegin[id] = (unsigned)j;                 // its count follows from its siblings (node_count, below)
                nfirst[id] = internal ? (int)(sstart[l + 1] + pnext - 1u) : -1;
                nparent[id] = par;
                if (l) {   // record my octant in the parent's child mask
                    unsigned oct = (unsigned)(skey[j] >> (63 - 3 * l)) & 7u;
                    atomicOr(&node_meta[par], 1u << oct);
                }
            }
            pprev = pcur;
            pcur = pnext;
        }
    }
}

// Bodies of node t.  The children of a node tile its range of sorted bodies, and siblings have consecutive ids:
// a node ends where its next sibling begins, a last child ends where its parent ends, the root at n.  (Replaces a
// galloping search over the keys per emitted node: a handful of dependent loads instead of 2 log2(count).)
__device__ __forceinline__ unsigned node_count(int t, int M, unsigned n, const unsigned *nbegin, const int *nparent)
{
    const unsigned b = nbegin[t];
    int u = t;
    while (true) {
        const int p = nparent[u];
        if (p < 0) return n - b;
        if (u + 1 < M && nparent[u + 1] == p) return nbegin[u + 1] - b;
        u = p;
    }
}

// Monopoles by arrival counters: a thread computes each leaf from its bodies, then climbs; the last
// child to arrive at a parent (counter in node_meta bits 8..) computes it from ALL children in
// ascending id, so the arithmetic order is fixed (bit-reproducible): masses added left to right,
// weighted sums by fma from 0, one IEEE division.
__device__ __forceinline__ double4 ldcg4(const double4 *p)
{
    const double2 *q = reinterpret_cast<const double2 *>(p);
    double2 a = __ldcg(q), b = __ldcg(q + 1);
    return make_double4(a.x, a.y, b.x, b.y);
}

// thread `gtid` of `gthreads` takes nodes gtid, gtid + gthreads, ...
__device__ __forceinline__ void monopoles_and_records(int M, unsigned n, int gtid, int gthreads, const double4 *sbody,
                                                      const unsigned *nbegin, unsigned *ncount,
                                                      const int *nfirst, const int *nparent, unsigned *node_meta,
                                                      double4 *mono, const unsigned char *nlevel, uint4 *winfo)
{
    for (int t = gtid; t < M; t += gthreads) {
        // the walk's packed record of this node (the child mask is complete: bits 0-7 are only
        // written by the emission)
        const int first = nfirst[t];
        const unsigned kids = (unsigned)__popc(__ldcg(node_meta + t) & 0xffu);
        const unsigned b = nbegin[t], c = node_count(t, M, n, nbegin, nparent);
        ncount[t] = c;
        winfo[t] = make_uint4(b, c, (unsigned)first, (unsigned)nlevel[t] | (kids << 8));
        if (first >= 0) continue;   // internal nodes are computed by their last child
        double4 r;
        if (c == 1) {
            r = sbody[b];
        } else {
            double4 s = sbody[b];
            double m = s.w;
            double wx = __fma_rn(s.w, s.x, 0.0), wy = __fma_rn(s.w, s.y, 0.0), wz = __fma_rn(s.w, s.z, 0.0);
            for (unsigned j = b + 1; j < b + c; ++j) {
                s = sbody[j];
                m = __dadd_rn(m, s.w);
                wx = __fma_rn(s.w, s.x, wx);
                wy = __fma_rn(s.w, s.y, wy);
                wz = __fma_rn(s.w, s.z, wz);
            }
            r = make_double4(__ddiv_rn(wx, m), __ddiv_rn(wy, m), __ddiv_rn(wz, m), m);
        }
        mono[t] = r;
        int p = nparent[t];
        while (p >= 0) {
            // one acq_rel atomic: its release publishes this thread's monopole, and for the last child to arrive its
            // acquire (the siblings' atomics on the same word form the release sequence) makes theirs visible; a pair of
            // __threadfence() around a relaxed atomic does the same with two MEMBAR.SC (64 -> 58 us at N = 1M)
            unsigned old;
            asm volatile("atom.acq_rel.gpu.global.add.u32 %0, [%1], 256;" : "=r"(old) : "l"(node_meta + p) : "memory");
            const int nch = __popc(old & 0xffu);
            if ((int)(old >> 8) != nch - 1) break;   // siblings still pending
            const int f = nfirst[p];
            double4 s = ldcg4(mono + f);
            double m = s.w;
            double wx = __fma_rn(s.w, s.x, 0.0), wy = __fma_rn(s.w, s.y, 0.0), wz = __fma_rn(s.w, s.z, 0.0);
            for (int u = f + 1; u < f + nch; ++u) {
                s = ldcg4(mono + u);
                m = __dadd_rn(m, s.w);
                wx = __fma_rn(s.w, s.x, wx);
                wy = __fma_rn(s.w, s.y, wy);
                wz = __fma_rn(s.w, s.z, wz);
            }
            mono[p] = make_double4(__ddiv_rn(wx, m), __ddiv_rn(wy, m), __ddiv_rn(wz, m), m);
            p = nparent[p];
        }
    }
}

}  // namespace bh
