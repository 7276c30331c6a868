// bh_common.cuh — shared declarations of the CUDA path (device state, workspace layout, launchers).
// Nothing here is shared with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <atomic>

#include "bh.h"

namespace bh {

constexpr int kMaxLevel = BH_MAX_LEVEL;   // 21
constexpr int kLevels = kMaxLevel + 1;    // levels 0..21
constexpr int kMaxGroup = 32;             // W <= 32: a walk group is evaluated by one warp (run-time, bh_create)
constexpr int kMaxGroupCell = 2048;       // Gc <= 2048 (run-time, bh_set_group_cell): bounds the window scratch of the tree kernels
constexpr int kMaxBboxBlocks = 1024;       // rows of the bounding-box partials
constexpr int kDefaultSMs = 148;          // B200; the real count is queried once per device (sm_count())
constexpr int kRadixBits = 8;
constexpr int kRadix = 1 << kRadixBits;   // 256 bins
constexpr int kSortPasses = 8;            // 63 key bits
constexpr int kSortThreads = 256;
constexpr int kSortItems = 16;              // keys per thread
constexpr int kSortTile = kSortThreads * kSortItems;   // 4096 keys per tile (one tile: the one-block build, bh_small.cu)
constexpr int64_t kSortSmallTileBelow = 1 << 19;   // the streaming passes use 2048-key tiles below this many keys
constexpr int kTreeTile = 1024;           // bodies per block in the tree kernels
constexpr int kDiagBlocks = 592;          // diagnostics: a FIXED number of partial sums, whatever the device, so that the reduction order is fixed
constexpr int kStackSlab = 22 * 256;      // walk: spill entries (8 bytes each) per producer warp: <= 32 x 7 ranges per level; overflow sets kStatStack

enum StatusBits : int { kStatNonFinite = 1, kStatCapacity = 2, kStatStack = 4, kStatRange = 8, kStatBpStack = 16,
                        kStatLongRun = 32 /* internal to the one-kernel sort: not an error, cleared by it */ };
constexpr int kMaxExtentExp = 300;        // largest extent must lie in [2^-300, 2^300] (or be 0): bh.h preconditions
constexpr int kNumStats = BH_NUM_STATS;

// Device-resident state of one build; written by kernels, read by later kernels (no host round trip).
struct DevState {
    double lo[3];          // cube corner
    double side;           // L = 2^e
    double scale;          // 2^(21-e)
    int e;                 // exponent of L
    int status;            // StatusBits, OR-ed by kernels, cleared by the host once it has reported them
    int n_nodes;           // M
    int depth;             // deepest level
    unsigned n_groups;     // Ng walk groups
    unsigned lvl_start[kLevels + 1];   // first node id of each level (lvl_start[kLevels] = M)
    unsigned ticket_bbox;  // last-block election
    unsigned walk_queue;   // dynamic group counter of the walk (reset by the walk's last producer warp)
    unsigned walk_done;    // producer warps that have left the walk
    unsigned ticket_diag;  // last-block election of the diagnostics reduction (resets itself)
    unsigned mid_bar[4];   // two grid barriers of the one-kernel build of mid-size sets (arrivals, generation; they reset themselves)
    unsigned long long pair_count;     // broad phase: candidate pairs found (may exceed the caller's capacity)
    unsigned long long agg_counts[3];  // aggregates: connected components, aggregates (size > 1), bad pairs
    unsigned long long stats[kNumStats];   // n_mono, n_direct, interactions, nodes tested, stack spills
};

// Pointers into the caller's workspace.
struct Workspace {
    DevState *st;
    double *bbox_part;        // [bbox blocks][6]
    unsigned *zero_begin;     // start of the region cleared at every build
    unsigned *hist;           // [kSortPasses][256]
    unsigned *sort_ticket;    // [kSortPasses]
    unsigned *lookback;       // [kSortPasses][tiles][256]
    unsigned *node_meta;      // [cap] bits 0-7 child mask, bits 8.. arrival counter
    size_t zero_bytes;
    unsigned long long *key[2];   // [n] double buffer
    unsigned *idx[2];             // [n]
    unsigned *iperm;              // [n] original index -> sorted position
    double4 *sbody;               // [n] sorted (x,y,z,m)
    unsigned *gstart;             // [Ng+1] first sorted body of each walk group (capacity n+1)
    double *gbox;                 // [Ng][6] lo xyz, hi xyz (capacity n)
    uchar4 *dlev;                 // [n] (first level this body starts a node at, its leaf level, group-start flag, group-cell level)
    unsigned *tile_lvl;           // [kLevels+1][tree tiles] per-tile node counts (+ group starts), then exclusive bases
    // nodes, SoA, ids in level/Morton order
    unsigned char *nlevel;
    unsigned *nbegin;
    unsigned *ncount;
    int *nfirst;
    int *nparent;
    double4 *mono;
    uint4 *winfo;                 // [M] walk record: begin, count, first_child, level | children << 8
    unsigned *cnt_mono;           // [Ng] (capacity n)
    unsigned *cnt_direct;         // [Ng]
    unsigned *walk_stack;         // [walk producer warps][kStackSlab][2]
    double *acc;                  // [n][3] internal accelerations (KDK state, host staging)
    double *stage_pos;            // [n][3] host-call staging; also the direct kernel's partial sums
    int64_t stage_doubles;        // capacity of stage_pos in doubles
    double *stage_mass;           // [n]
    double *diag_part;            // [kDiagBlocks][8][2] double-double partial sums of the diagnostics
    double *diag_out;             // [8] conserved quantities, [8] bits of the Eq. (7) maximum
    unsigned *diag_ticket;        // = &st->ticket_diag
    // rows NEXT-3 / NEXT-4 (bh_contact.cu)
    double *bsort;                // [n] bounding radius b of the sorted bodies
    double4 *box_lo;              // [cap] per node: min x,y,z of its bodies' centres, max b
    double4 *box_hi;              // [cap] per node: max x,y,z
    unsigned *bp_cnt;             // [cap] arrival counters of the node-box pass
    int *agg_size;                // [n] component sizes when the caller wants none
    int64_t node_cap;
    int64_t sort_tiles;
    int64_t tree_tiles;
    int walk_warps;               // producer warps of the walk = SMs x pairs per block
    int sms;                      // multiprocessors of the device (grid sizing)
    int leaf_cap;                 // C
    int group_w;                  // W, bodies per walk group (1..32)
    int group_cell;               // Gc
    size_t total_bytes;
};

struct WalkConfig {
    static constexpr int kPairsPerBlock = 8;   // producer/consumer warp pairs in the one block of an SM
};

// multiprocessors of the current device, queried once per device; kDefaultSMs when there is no device (host-only
// argument checks and size queries still work)
int sm_count();
// ordinal of the current CUDA device, 0 when there is none; below kMaxDevices.  What a launcher sets up once
// (shared-memory attributes, occupancy, cooperative-launch support) it sets up once PER DEVICE, indexed by this.
constexpr int kMaxDevices = 64;
int current_device();

inline int64_t node_capacity(int64_t n, int leaf_cap) { return n + 21 * (n / (leaf_cap + 1)) + 1; }

// carve the workspace; base may be nullptr to compute the size only
Workspace carve(char *base, int64_t max_n, int leaf_cap);

// launchers (each enqueues on `s`)
void launch_cube(const Workspace &w, const double *pos, int64_t n, cudaStream_t s);
void launch_keys(const Workspace &w, const double *pos, int64_t n, cudaStream_t s);
int launch_sort(const Workspace &w, const double *pos, int64_t n, cudaStream_t s);   // result in key[0]/idx[0]; returns the launches
int sort_tile_items(int64_t n);                                    // keys per thread of the streaming passes for n keys
// steps a1-a6 in one kernel of one block, n <= kSortTile (bh_small.cu); needs no prior clearing
void launch_build_small(const Workspace &w, const double *pos, const double *mass, int64_t n, cudaStream_t s);
// steps a1-a6 in one co-resident kernel with grid barriers, kSortTile < n <= mid_build_limit (bh_mid.cu); needs no prior
// clearing; returns the launches (1) or -1 if the cooperative launch was refused
int64_t mid_build_limit(const Workspace &w);
int launch_build_mid(const Workspace &w, const double *pos, const double *mass, int64_t n, cudaStream_t s);
// sorted bodies AND group boxes in one pass, after launch_tree (which then only builds the tree from the keys)
void launch_gather_boxes(const Workspace &w, const double *pos, const double *mass, int64_t n, cudaStream_t s);
// (x,y,z,m) in the caller's body order with the identity permutation: input of a direct sum without a tree
void launch_pack(const Workspace &w, const double *pos, const double *mass, int64_t n, cudaStream_t s);
void launch_iperm(const Workspace &w, int64_t n, cudaStream_t s);   // w.iperm from the permutation of the last build
void launch_tree(const Workspace &w, int64_t n, int leaf_cap, cudaStream_t s);
void launch_monopoles(const Workspace &w, int64_t n, cudaStream_t s);
// mode 0: acc [n][3] accelerations; 1: acc [n] potential; 2: acc [n][3] and phi [n] from one walk (NEXT-1)
void launch_walk(const Workspace &w, int64_t n, double theta, double eps, double G, double *acc, int mode, double *phi,
                 cudaStream_t s);
int launch_direct(const Workspace &w, int64_t n, const int32_t *tgt, int64_t nt, double eps, double G,
                  double *acc, bool potential, cudaStream_t s);   // returns the number of kernels launched
void launch_kick_drift(double *pos, double *vel, const double *acc, int64_t n, double dt, cudaStream_t s);
// the same update and, in the same pass, step a1 for the new positions (the build that follows skips launch_cube)
void launch_kick_drift_cube(const Workspace &w, double *pos, double *vel, const double *acc, int64_t n, double dt,
                            cudaStream_t s);
void launch_kick(double *vel, const double *acc, int64_t n, double h, cudaStream_t s);
void launch_unpack_mask(const Workspace &w, unsigned char *mask_out, int64_t cap, cudaStream_t s);
// rows "next" (bh_diag.cu): results land in w.diag_out
void launch_diagnostics(const Workspace &w, const double *pos, const double *vel, const double *mass,
                        const double *phi, int64_t n, cudaStream_t s);
void launch_position_error(const Workspace &w, const double *pos, const double *ref, int64_t n, cudaStream_t s);
// rows NEXT-3 / NEXT-4 (bh_contact.cu); each returns the number of kernels launched
int launch_broadphase(const Workspace &w, int64_t n, const double *radius, const double *vel, double dt,
                      int32_t *pairs, int64_t cap, cudaStream_t s);   // count lands in st->pair_count
int launch_aggregates(const Workspace &w, int64_t n, const int32_t *pairs, int64_t n_pairs, const double *mass_in,
                      int32_t *label, int32_t *size, double *mass, cudaStream_t s);   // counts in st->agg_counts
// record the message of a context-free call that failed; bh_last_error(NULL) returns it (per host thread)
void set_global_error(const char *msg);
void launch_euler_sub(double *pos, double *vel, const double *acc, int64_t n, double dt, int n_sub, cudaStream_t s);

// ---- small device helpers ----
__device__ __forceinline__ unsigned lane_id() { return threadIdx.x & 31u; }

// common leading 3-bit digits of two 63-bit keys (bit 63 is 0 in both): 0..21
__device__ __forceinline__ int common_levels(unsigned long long a, unsigned long long b)
{
    unsigned long long x = a ^ b;
    if (x == 0ull) return kMaxLevel;
    return (__clzll((long long)x) - 1) / 3;
}

}  // namespace bh
