// bh_tree.cuh — block-level bodies of steps a4-a6 (group boxes, octree from the sorted keys, monopoles), shared by
// the streaming kernels of bh_tree.cu (one call per thread block) and the one-block build of small body sets
// (bh_small.cu: the same functions called for every tile in turn).  See bh_tree.cu for the derivation.
// Pointers to data that the build itself produces are NOT const __restrict__ here: in the one-block build a phase
// reads what an earlier phase of the same kernel wrote, which must not go through the non-coherent load path.
#pragma once
#include "bh_common.cuh"

namespace bh {

// exact bounding box of every walk group: warp `wid` of `nwarps` takes groups wid, wid + nwarps, ...
__device__ __forceinline__ void group_boxes(unsigned ng, unsigned wid, unsigned nwarps, const unsigned *gstart,
                                            const double4 *sbody, double *gbox)
{
    const unsigned lane = lane_id();
    const double inf = __longlong_as_double(0x7ff0000000000000ll);
    for (unsigned g = wid; g < ng; g += nwarps) {
        const unsigned b = gstart[g], e = gstart[g + 1];
        double lx = inf, ly = inf, lz = inf, hx = -inf, hy = -inf, hz = -inf;
        for (unsigned j = b + lane; j < e; j += 32) {
            const double4 p = sbody[j];
            lx = fmin(lx, p.x); ly = fmin(ly, p.y); lz = fmin(lz, p.z);
            hx = fmax(hx, p.x); hy = fmax(hy, p.y); hz = fmax(hz, p.z);
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            lx = fmin(lx, __shfl_xor_sync(0xffffffffu, lx, o));
            ly = fmin(ly, __shfl_xor_sync(0xffffffffu, ly, o));
            lz = fmin(lz, __shfl_xor_sync(0xffffffffu, lz, o));
            hx = fmax(hx, __shfl_xor_sync(0xffffffffu, hx, o));
            hy = fmax(hy, __shfl_xor_sync(0xffffffffu, hy, o));
            hz = fmax(hz, __shfl_xor_sync(0xffffffffu, hz, o));
        }
        if (lane == 0) {
            double *q = gbox + 6ull * g;
            q[0] = lx; q[1] = ly; q[2] = lz; q[3] = hx; q[4] = hy; q[5] = hz;
        }
    }
}

// sliding maximum over windows of k consecutive entries of a[0..len): after the call a[i] holds
// max(a[i .. i+2^p-1]) with p = floor(log2 k); the caller combines a[i] and a[i + k - 2^p].
__device__ __forceinline__ int window_doubling(signed char *a, int len, int k)
{
    int p = 0;
    while ((2 << p) <= k) ++p;
    for (int r = 0; r < p; ++r) {
        const int h = 1 << r;
        signed char v[12];   // len <= kTreeTile + kMaxGroupCell, >= 256 threads
        int c = 0;
        for (int i = threadIdx.x; i < len; i += blockDim.x, ++c) {
            signed char x = a[i];
            if (i + h < len) x = max(x, a[i + h]);
            v[c] = x;
        }
        __syncthreads();
        c = 0;
        for (int i = threadIdx.x; i < len; i += blockDim.x, ++c) a[i] = v[c];
        __syncthreads();
    }
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

// Tile `tile` of kTreeTile bodies, any block size >= 256: per body (d+1, leaf, group-start flag, group-cell level) and the
// tile's counts of nodes per level and of group starts.  sw: kTreeTile + C + kTreeTile + Gc bytes of shared
// memory; shist: kLevels + 1 words.
__device__ __forceinline__ void tree_levels_tile(const unsigned long long *skey, long long n, int C, int Gc, int W,
                                                 uchar4 *dlev, unsigned *tile_lvl, int ntiles, int tile,
                                                 signed char *sw, unsigned *shist)
{
    signed char *swc = sw;
    signed char *swg = sw + kTreeTile + C;
    const long long t0 = (long long)tile * kTreeTile;
    if (threadIdx.x <= kLevels) shist[threadIdx.x] = 0u;
    for (int k = threadIdx.x; k < kTreeTile + C; k += blockDim.x) {
        long long s = t0 - C + k;
        int wv = -1;
        if (s >= 0 && s + C < n) wv = common_levels(skey[s], skey[s + C]);
        swc[k] = (signed char)wv;
    }
    for (int k = threadIdx.x; k < kTreeTile + Gc; k += blockDim.x) {
        long long s = t0 - Gc + k;
        int wv = -1;
        if (s >= 0 && s + Gc < n) wv = common_levels(skey[s], skey[s + Gc]);
        swg[k] = (signed char)wv;
    }
    __syncthreads();
    const int pc = window_doubling(swc, kTreeTile + C, C + 1);
    const int pg = window_doubling(swg, kTreeTile + Gc, Gc + 1);
    for (int k = threadIdx.x; k < kTreeTile; k += blockDim.x) {
        long long j = t0 + k;
        if (j >= n) break;
        // windows of C+1 (Gc+1) bodies that start at j-C .. j  (j-Gc .. j)
        const int mw = max((int)swc[k], (int)swc[k + C + 1 - pc]);
        const int mg = max((int)swg[k], (int)swg[k + Gc + 1 - pg]);
        const int leaf = min(kMaxLevel, mw + 1);
        const int glev = min(leaf, mg + 1);
        const int d = (j == 0) ? -1 : common_levels(skey[j - 1], skey[j]);
        const unsigned cb = range_begin(skey, (unsigned)j, glev);
        const bool gs = (((unsigned)j - cb) % (unsigned)W) == 0u;
        dlev[j] = make_uchar4((unsigned char)(d + 1), (unsigned char)leaf, gs ? 1 : 0, (unsigned char)glev);
        for (int l = d + 1; l <= leaf; ++l) atomicAdd(&shist[l], 1u);
        if (gs) atomicAdd(&shist[kLevels], 1u);
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
                                               unsigned *ncount, int *nfirst, int *nparent, unsigned *node_meta,
                                               unsigned *gstart, unsigned (*scnt)[kLevels + 1], unsigned *sstart)
{
    constexpr int kChunks = kTreeTile / 32;          // 32 chunks of 32 bodies
    const unsigned lane = lane_id(), warp = threadIdx.x >> 5;
    const int nwarps = blockDim.x >> 5;
    const long long t0 = (long long)tile * kTreeTile;
    if (threadIdx.x <= kLevels) sstart[threadIdx.x] = st->lvl_start[threadIdx.x];
    if ((long long)st->n_nodes > node_cap) return;   // flagged by the scan; stay in bounds (uniform over the block)
    // phase 1: per chunk level counts
    for (int c = warp; c < kChunks; c += nwarps) {
        long long j = t0 + c * 32 + lane;
        uchar4 dl = j < n ? dlev[j] : make_uchar4(255, 0, 0, 0);
#pragma unroll
        for (int l = 0; l < kLevels; ++l) {
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
        // inclusive per-level counts at this body: prev (l-1), cur (l), next (l+1)
        unsigned pprev = 0, pcur, pnext;
        {
            unsigned b = __ballot_sync(0xffffffffu, first <= 0 && 0 <= leaf);
            pcur = scnt[c][0] + __popc(b & le);
        }
#pragma unroll 1
        for (int l = 0; l < kLevels; ++l) {
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
                nbegin[id] = (unsigned)j;
                ncount[id] = range_end(skey, (unsigned)n, (unsigned)j, l) - (unsigned)j;
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
__device__ __forceinline__ void monopoles_and_records(int M, int gtid, int gthreads, const double4 *sbody,
                                                      const unsigned *nbegin, const unsigned *ncount,
                                                      const int *nfirst, const int *nparent, unsigned *node_meta,
                                                      double4 *mono, const unsigned char *nlevel, uint4 *winfo)
{
    for (int t = gtid; t < M; t += gthreads) {
        // the walk's packed record of this node (the child mask is complete: bits 0-7 are only
        // written by the emission)
        const int first = nfirst[t];
        const unsigned kids = (unsigned)__popc(__ldcg(node_meta + t) & 0xffu);
        winfo[t] = make_uint4(nbegin[t], ncount[t], (unsigned)first, (unsigned)nlevel[t] | (kids << 8));
        if (first >= 0) continue;   // internal nodes are computed by their last child
        const unsigned b = nbegin[t], c = ncount[t];
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
            __threadfence();
            const unsigned old = atomicAdd(&node_meta[p], 256u);
            const int nch = __popc(old & 0xffu);
            if ((int)(old >> 8) != nch - 1) break;   // siblings still pending
            __threadfence();
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
