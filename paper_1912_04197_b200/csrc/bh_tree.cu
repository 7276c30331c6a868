// bh_tree.cu — steps a4 (gather to sorted (x,y,z,m) + group boxes), a5 (octree from sorted keys) and
// a6 (monopoles, Eq. (2), by atomic arrival counters).
//
// a5 is built WITHOUT a level loop.  With sorted keys, let
//     d_j    = number of leading 3-bit digits that key j shares with key j-1          (d_0 = -1)
//     w_s    = digits shared by keys s and s+C  (a window of C+1 bodies),  -1 if s+C >= n
//     leaf_j = min(21, 1 + max_{s in [j-C, j]} w_s)            (0 if no such window exists)
// A cell at level l containing body j holds more than C bodies iff some window of C+1 consecutive
// bodies around j shares l digits, i.e. iff l <= leaf_j - 1; so the canonical tree (R8,
// R9) has a node at (level l, first body j) exactly when  d_j < l <= leaf_j,  and that node is a leaf
// iff l == leaf_j.  Node ids are level-major and Morton-ordered inside a level, so
//     id(l, j) = lvl_start[l] + #{j' <= j : d_j' < l <= leaf_j'} - 1
// which is a per-level prefix count; parent and first child are the same count at levels l-1 and
// l+1.  Three streaming kernels: per-body (d, leaf) + per-tile level histograms; a scan of the tile
// histograms; emission.
//
// Walk groups (R6) come out of the same three kernels.  A GROUP CELL is a node holding <= Gc bodies
// (or a leaf) whose parent holds more than Gc; its level for body j is
//     glev_j = min(leaf_j, 1 + max_{s in [j-Gc, j]} (digits shared by keys s and s+Gc))
// and body j starts a group iff its distance to the first body of its group cell is a multiple of
// W.  Group starts are counted and ranked like one more "level" (row kLevels of the histograms).
#include "bh_tree.cuh"

namespace bh {

// ------------------------------------------------------------------------------------------ a4
// inverse permutation (body index -> sorted position), made only when a call needs it (bh_direct_targets): a
// scattered 4-byte store per body is not worth paying in every build
__global__ void __launch_bounds__(256) iperm_kernel(const unsigned *__restrict__ perm, long long n,
                                                    unsigned *__restrict__ iperm)
{
    const long long j = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (j < n) iperm[perm[j]] = (unsigned)j;
}

__global__ void __launch_bounds__(256) pack_kernel(const double *__restrict__ pos, const double *__restrict__ mass,
                                                   long long n, double4 *__restrict__ sbody,
                                                   unsigned *__restrict__ perm)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    sbody[i] = make_double4(pos[3 * i], pos[3 * i + 1], pos[3 * i + 2], mass[i]);
    perm[i] = (unsigned)i;
}

// a4 + group boxes in one pass (streaming build): the tree only needs the sorted keys, so the bodies are gathered AFTER
// it, a warp per walk group (at most 32 bodies: one per lane), and the group's box is reduced from the registers that
// are being stored — the sorted bodies are not read back for it (32 B per body less than gather + group_box_kernel).
__global__ void __launch_bounds__(256) gather_box_kernel(const DevState *__restrict__ st, const double *__restrict__ pos,
                                                         const double *__restrict__ mass,
                                                         const unsigned *__restrict__ perm,
                                                         const unsigned *__restrict__ gstart,
                                                         double4 *__restrict__ sbody, double *__restrict__ gbox)
{
    const unsigned lane = lane_id();
    const unsigned ng = st->n_groups;
    const unsigned nwarps = (gridDim.x * blockDim.x) >> 5;
    for (unsigned g = (blockIdx.x * blockDim.x + threadIdx.x) >> 5; g < ng; g += nwarps) {
        const unsigned b = gstart[g], e = gstart[g + 1];
        const double inf = __longlong_as_double(0x7ff0000000000000ll);
        double lx = inf, ly = inf, lz = inf, hx = -inf, hy = -inf, hz = -inf;
        for (unsigned j = b + lane; j < e; j += 32) {           // W <= 32: at most one body per lane; kept general
            const unsigned i = perm[j];
            double4 p;
            p.x = __ldg(pos + 3ll * i + 0);
            p.y = __ldg(pos + 3ll * i + 1);
            p.z = __ldg(pos + 3ll * i + 2);
            p.w = __ldg(mass + i);
            sbody[j] = p;
            lx = fmin(lx, p.x); ly = fmin(ly, p.y); lz = fmin(lz, p.z);
            hx = fmax(hx, p.x); hy = fmax(hy, p.y); hz = fmax(hz, p.z);
        }
        // min / max are exact and order-free: the box equals group_boxes' (lanes without a body hold the neutral values)
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

// ------------------------------------------------------------------------------------------ a5
// Kernel A: per body (d+1, leaf, group-start flag) and per-tile counts of nodes per level and of
// group starts.
__global__ void __launch_bounds__(256) tree_levels_kernel(const unsigned long long *__restrict__ skey,
                                                          long long n, int C, int Gc, int W, uchar4 *__restrict__ dlev,
                                                          unsigned *__restrict__ tile_lvl, int ntiles)
{
    extern __shared__ unsigned sw[];      // leaf windows, group windows (two copies each), cell starts
    __shared__ unsigned shist[kLevels + 1];
    tree_levels_tile(skey, n, C, Gc, W, dlev, tile_lvl, ntiles, blockIdx.x, sw, shist);
}

// Kernel B (one block): exclusive scan of the tile counts of each level, level starts, node count, depth.
__global__ void __launch_bounds__((kLevels + 1) * 32) tree_scan_kernel(unsigned *tile_lvl, int ntiles, DevState *st,
                                                                       long long node_cap, unsigned *gstart,
                                                                       unsigned n)
{
    __shared__ unsigned stot[kLevels + 1];
    tree_scan_block(tile_lvl, ntiles, st, node_cap, gstart, n, stot);
}

// Kernel C: emit the nodes.
__global__ void __launch_bounds__(256) tree_emit_kernel(const unsigned long long *__restrict__ skey, long long n,
                                                        const uchar4 *__restrict__ dlev,
                                                        const unsigned *__restrict__ tile_lvl, int ntiles,
                                                        const DevState *__restrict__ st, long long node_cap,
                                                        unsigned char *__restrict__ nlevel,
                                                        unsigned *__restrict__ nbegin,
                                                        int *__restrict__ nfirst, int *__restrict__ nparent,
                                                        unsigned *node_meta, unsigned *__restrict__ gstart)
{
    __shared__ unsigned scnt[kTreeTile / 32][kLevels + 1];  // per chunk, per level (+ group starts): counts -> bases
    __shared__ unsigned sstart[kLevels + 1];
    tree_emit_tile(skey, n, dlev, tile_lvl, ntiles, blockIdx.x, st, node_cap, nlevel, nbegin, nfirst, nparent,
                   node_meta, gstart, scnt, sstart);
}

// ------------------------------------------------------------------------------------------ a6
__global__ void __launch_bounds__(256) monopole_kernel(const DevState *__restrict__ st, unsigned n,
                                                       const double4 *__restrict__ sbody,
                                                       const unsigned *__restrict__ nbegin,
                                                       unsigned *__restrict__ ncount,
                                                       const int *__restrict__ nfirst,
                                                       const int *__restrict__ nparent, unsigned *node_meta,
                                                       double4 *mono, long long node_cap,
                                                       const unsigned char *__restrict__ nlevel,
                                                       uint4 *__restrict__ winfo)
{
    const int M = st->n_nodes;
    if ((long long)M > node_cap) return;
    monopoles_and_records(M, n, blockIdx.x * blockDim.x + threadIdx.x, gridDim.x * blockDim.x, sbody, nbegin, ncount, nfirst,
                          nparent, node_meta, mono, nlevel, winfo);
}

__global__ void unpack_mask_kernel(const unsigned *__restrict__ node_meta, const DevState *__restrict__ st,
                                   unsigned char *__restrict__ out, long long cap)
{
    const long long M = st->n_nodes < cap ? st->n_nodes : cap;
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < M;
         t += (long long)gridDim.x * blockDim.x)
        out[t] = (unsigned char)(node_meta[t] & 0xffu);
}

// ------------------------------------------------------------------------------------------ launchers
void launch_iperm(const Workspace &w, int64_t n, cudaStream_t s)
{
    iperm_kernel<<<(int)((n + 255) / 256), 256, 0, s>>>(w.idx[0], n, w.iperm);
}

void launch_pack(const Workspace &w, const double *pos, const double *mass, int64_t n, cudaStream_t s)
{
    pack_kernel<<<(int)((n + 255) / 256), 256, 0, s>>>(pos, mass, n, w.sbody, w.idx[0]);
}

void launch_tree(const Workspace &w, int64_t n, int leaf_cap, cudaStream_t s)
{
    const int ntiles = (int)((n + kTreeTile - 1) / kTreeTile);
    size_t smem = (size_t)tree_levels_smem_words(leaf_cap, w.group_cell) * sizeof(unsigned);
    tree_levels_kernel<<<ntiles, 256, smem, s>>>(w.key[0], n, leaf_cap, w.group_cell, w.group_w, w.dlev, w.tile_lvl, ntiles);
    tree_scan_kernel<<<1, (kLevels + 1) * 32, 0, s>>>(w.tile_lvl, ntiles, w.st, w.node_cap, w.gstart, (unsigned)n);
    tree_emit_kernel<<<ntiles, 256, 0, s>>>(w.key[0], n, w.dlev, w.tile_lvl, ntiles, w.st, w.node_cap, w.nlevel,
                                            w.nbegin, w.nfirst, w.nparent, w.node_meta, w.gstart);
}

// sorted bodies + group boxes, after launch_tree (needs the group starts)
void launch_gather_boxes(const Workspace &w, const double *pos, const double *mass, int64_t n, cudaStream_t s)
{
    int64_t want = (n + 7) / 8;                   // about a warp per 32 bodies, eight warps per block
    int blocks = (int)(want < (int64_t)w.sms * 32 ? want : (int64_t)w.sms * 32);
    if (blocks < 1) blocks = 1;
    gather_box_kernel<<<blocks, 256, 0, s>>>(w.st, pos, mass, w.idx[0], w.gstart, w.sbody, w.gbox);
}

void launch_monopoles(const Workspace &w, int64_t n, cudaStream_t s)
{
    const int64_t want = (node_capacity(n, w.leaf_cap) + 255) / 256;
    int blocks = (int)(want < w.sms * 16 ? want : w.sms * 16);
    monopole_kernel<<<blocks, 256, 0, s>>>(w.st, (unsigned)n, w.sbody, w.nbegin, w.ncount, w.nfirst, w.nparent, w.node_meta,
                                           w.mono, w.node_cap, w.nlevel, w.winfo);
}

void launch_unpack_mask(const Workspace &w, unsigned char *mask_out, int64_t cap, cudaStream_t s)
{
    unpack_mask_kernel<<<w.sms * 4, 256, 0, s>>>(w.node_meta, w.st, mask_out, cap);
}

}  // namespace bh
