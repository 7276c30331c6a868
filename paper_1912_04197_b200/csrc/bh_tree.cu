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
__global__ void __launch_bounds__(256) gather_kernel(const double *__restrict__ pos,
                                                     const double *__restrict__ mass,
                                                     const unsigned *__restrict__ perm, long long n,
                                                     double4 *__restrict__ sbody)
{
    const long long j = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= n) return;
    const unsigned i = perm[j];
    double4 b;
    b.x = __ldg(pos + 3ll * i + 0);
    b.y = __ldg(pos + 3ll * i + 1);
    b.z = __ldg(pos + 3ll * i + 2);
    b.w = __ldg(mass + i);
    sbody[j] = b;
}

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

__global__ void __launch_bounds__(256) group_box_kernel(const DevState *__restrict__ st,
                                                        const unsigned *__restrict__ gstart,
                                                        const double4 *__restrict__ sbody,
                                                        double *__restrict__ gbox)
{
    group_boxes(st->n_groups, (blockIdx.x * blockDim.x + threadIdx.x) >> 5, (gridDim.x * blockDim.x) >> 5, gstart, sbody, gbox);
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
void launch_gather(const Workspace &w, const double *pos, const double *mass, int64_t n, cudaStream_t s)
{
    int blocks = (int)((n + 255) / 256);
    gather_kernel<<<blocks, 256, 0, s>>>(pos, mass, w.idx[0], n, w.sbody);
}

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
    group_box_kernel<<<w.sms * 4, 256, 0, s>>>(w.st, w.gstart, w.sbody, w.gbox);
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
