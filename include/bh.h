/*
 * bh.h — C ABI of libbh: fp64 Barnes-Hut mutual gravity on one NVIDIA B200 (sm_100a).
 *
 * The library implements the data-parallel hot path of arxiv/paper_1912_04197 (Ferrari, Lavagna &
 * Blazquez): the gravity module of PAPER.md §2.1 (lines 45-118).  Every step runs in hand-written
 * CUDA kernels; there is no CPU fallback.  Citations are PAPER.md:<line>; "R<k>" are the readings
 * of the paper listed in DESIGN.md §3.
 *
 * Conventions
 *   - Pointers named *_dev are CUDA device pointers, *_host are host pointers.  fp64 throughout
 *     ("full double precision").  Arrays are dense, row-major: pos/vel/acc are [n][3].
 *   - Every call enqueues its work on the context's stream and returns without waiting for the
 *     GPU, except the calls documented as synchronising (bh_synchronize, bh_eval_host and the
 *     bh_get_* calls marked so below).  A context is not thread-safe.
 *   - Return value: BH_OK (0) or a negative bh_status.  No exceptions, no abort().  Data errors that
 *     only the GPU can see (non-finite coordinates, node capacity) are sticky: they are reported by
 *     the next synchronising call.  bh_last_error() gives a human-readable message.
 *   - Devices: a context belongs to the CUDA device that was current at bh_create (its workspace, stream and
 *     events live there).  Make that device current before every call on the context; a call that touches the
 *     GPU with another device current returns BH_ERR_STATE.  One process may hold contexts on several devices;
 *     what the library sets up once per kernel (shared-memory limits, occupancy) it sets up per device.
 *     bh_last_error(NULL) returns the message of the last context-free call that failed on this host thread
 *     (bh_create, bh_diagnostics_static).
 *   - Ownership: the caller owns every buffer it passes, including the workspace; the library
 *     allocates no device memory except a few bytes of pinned host memory at bh_create.
 *   - Range of the input.  Checked on the GPU (sticky BH_ERR_NONFINITE / BH_ERR_INVALID_ARG): every
 *     coordinate finite; the largest extent E = max over axes of (max - min) either 0 or in
 *     [2^-300, 2^300] (the squares of cell edges and distances that the opening test compares, Eq. (3)
 *     PAPER.md:86, then stay normal doubles down to level 21).  Not checked: masses finite and > 0 (R15),
 *     and such that m x (Eq. (2)) and m / r^3 (Eq. (6)) are representable for the coordinates and
 *     distances that occur.  A pair whose softened squared
 *     distance |d|^2 + eps^2 is below the smallest normal double (2.2e-308; eps = 0 with coincident
 *     bodies is the usual case) contributes nothing (R13).
 */
#ifndef BH_H_
#define BH_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct bh_ctx bh_ctx; /* opaque */

typedef enum {
    BH_OK = 0,
    BH_ERR_INVALID_ARG = -1, /* null pointer, n < 1, n > max_n, leaf_cap < 1, theta < 0, eps < 0, ... */
    BH_ERR_CAPACITY = -2,    /* workspace too small / node array overflow */
    BH_ERR_NONFINITE = -3,   /* a coordinate is NaN or infinite (found by the bounding-box reduction) */
    BH_ERR_STATE = -4,       /* call order: accel/direct before build, kdk_step before bind_state */
    BH_ERR_CUDA = -5         /* a CUDA runtime call or an earlier asynchronous launch failed */
} bh_status;

#define BH_MAX_LEVEL 21    /* 63-bit Morton keys, 3 bits per level (R9) */
/* Reading R6: W bodies walk the tree together (bh_create group_size, default 32),
 * and a group never straddles a tree cell that holds <= Gc bodies (bh_set_group_cell).  Both are parameters
 * of the method: the oracle takes them as arguments too, and parity is tested at several (W, Gc). */
#define BH_GROUP_SIZE_DEFAULT 32
#define BH_GROUP_CELL_DEFAULT 512
#define BH_NUM_STATS 5

/* Bytes of device workspace a context for up to max_n bodies needs.  0 if the arguments are invalid
 * (max_n < 1 or > 2^30, leaf_cap < 1 or > 1024, group_size < 0 or > 32).  Depends on the number of
 * multiprocessors of the current CUDA device: query it on the device the context will be created on. */
size_t bh_workspace_bytes(int64_t max_n, int leaf_cap, int group_size);

/* Create a context.  leaf_cap = C: a node is a leaf iff it holds <= C bodies or sits at level 21
 * (PAPER.md:62 subdivides "until each node ... contains zero or one particle" = C 1; R8).
 * group_size = W, the most bodies that walk the tree together: 1..32, 0 = 32 (R6).  W = 1 is the paper's
 * own per-body walk ("for each body-node pair", 118 "each body is assigned to a thread"): one warp
 * per body, slow, there to quantify the group reading against it.  workspace_dev must hold
 * bh_workspace_bytes() bytes, be 256-byte aligned and stay valid until bh_destroy.  cuda_stream is a
 * cudaStream_t (NULL = the legacy default stream). */
bh_status bh_create(bh_ctx **out, int64_t max_n, int leaf_cap, int group_size, void *workspace_dev,
                    size_t workspace_bytes, void *cuda_stream);
bh_status bh_destroy(bh_ctx *ctx);
bh_status bh_set_stream(bh_ctx *ctx, void *cuda_stream);

/* Group-cell capacity Gc of reading R6, 1..2048 (default BH_GROUP_CELL_DEFAULT): a group cell is a tree node
 * holding <= Gc bodies (or a leaf) whose parent holds more; group cells tile the sorted bodies and each is cut
 * into runs of W.  Takes effect at the next build. */
bh_status bh_set_group_cell(bh_ctx *ctx, int group_cell);

/* Build the octree of the n bodies ("re-built at each time step"):
 * bounding cube -> 63-bit Morton keys -> stable LSD radix sort -> sorted (x,y,z,m) bodies and group
 * boxes -> nodes (level, begin, count, first_child, child_mask, parent) in level/Morton order ->
 * monopoles, Eq. (2) PAPER.md:76.  pos_dev [n][3] and mass_dev [n] are read only and need not outlive
 * the call's execution on the stream. */
bh_status bh_build(bh_ctx *ctx, const double *pos_dev, const double *mass_dev, int64_t n);

/* Barnes-Hut accelerations of all bodies of the last build, Eqs. (3)-(6) PAPER.md:84-106, written
 * to acc_dev [n][3] in the body order given to bh_build.  theta >= 0 is the opening parameter
 * (cell edge / distance, R4; strict <, R5), eps >= 0 the Plummer softening of Eq. (6), G the
 * gravitational constant.  Output is acceleration, not force (R1). */
bh_status bh_accel(bh_ctx *ctx, double theta, double eps, double G, double *acc_dev);

/* Direct N^2 sum, Eq. (1), over the bodies of the last build; same softened kernel. */
bh_status bh_direct(bh_ctx *ctx, double eps, double G, double *acc_dev);

/* Direct sum for nt target bodies tgt_dev[k] (indices in bh_build order) against all n sources;
 * acc_dev is [nt][3].  For sampled checks at sizes where N^2 is too long. */
bh_status bh_direct_targets(bh_ctx *ctx, const int32_t *tgt_dev, int64_t nt, double eps, double G,
                            double *acc_dev);

/* Leapfrog kick-drift-kick (PAPER.md:148 lists leapfrog among the symplectic steppers; R18).
 * bh_bind_state borrows pos_dev/vel_dev [n][3] (updated IN PLACE by every step) and mass_dev [n].
 * bh_kdk_step(dt):  v += a dt/2;  x += v dt;  rebuild tree;  a = accel(x);  v += a dt/2, with
 * v = fma(a, dt/2, v) and x = fma(v, dt, x).  The first step after bind evaluates a(x0) once. */
bh_status bh_bind_state(bh_ctx *ctx, double *pos_dev, double *vel_dev, const double *mass_dev,
                        int64_t n, double theta, double eps, double G);
bh_status bh_kdk_step(bh_ctx *ctx, double dt);
/* Device pointer to the accelerations [n][3] held by the bound state (valid after a step). */
bh_status bh_get_state_acc(bh_ctx *ctx, const double **acc_dev);
/* Copy the accelerations [n][3] of the last evaluation a stepper made (bh_kdk_step: a(x) at the new
 * positions; bh_euler_step / bh_multirate_step: a(x_k) at the positions the step started from) into
 * acc_dev.  BH_ERR_STATE before the first step. */
bh_status bh_copy_state_acc(bh_ctx *ctx, double *acc_dev);

/* ---- rows "next" of SURVEY.md 8(f): the paper's stepping variants and conservation diagnostics ---- */

/* How the steppers (bh_kdk_step, bh_euler_step, bh_multirate_step) evaluate gravity
 * "through N^2 interactions or by building the octree" (direct for few bodies, octree for
 * many): method 0 = Barnes-Hut tree (default), 1 = direct N^2 sum, Eq. (1), without building a tree.
 * After a direct evaluation the context holds no tree: bh_accel etc. need a new bh_build. */
bh_status bh_set_gravity_method(bh_ctx *ctx, int method);

/* Replay the steppers through a CUDA graph (enable != 0).  A step at small N is bound by its kernel
 * launches (sixteen in a streaming build) (the paper sees the same: octree creation dominates for few bodies); with
 * the graph on, the second bh_kdk_step / bh_euler_step / bh_multirate_step call with the same arguments on
 * the same bound state is captured while it is enqueued and later calls replay it with one launch.
 * Results are bit-identical to the plain path.  Ignored while bh_set_timing is on (events are not
 * captured).  Any change of arguments, state or method simply captures again.  Measured on B200: the
 * host-side launch cost goes away, the step time does not change (0.155 ms at N = 10 either way) — the
 * dependent kernels' own latencies, not the launch rate, bound a small step. */
bh_status bh_set_graph(bh_ctx *ctx, int enable);

/* Semi-implicit (symplectic) Euler, the paper's preferred stepper, on the state of
 * bh_bind_state:  rebuild tree;  a = accel(x_k);  v_k+1 = fma(a, dt, v_k);  x_k+1 = fma(v_k+1, dt, x_k).
 * One evaluation per step.  Afterwards the context holds a(x_k), so a following bh_kdk_step starts by
 * evaluating a(x) again. */
bh_status bh_euler_step(bh_ctx *ctx, double dt);

/* Two-rate stepping, PAPER.md:338-340 ("we advance the simulation of dt_c ... but we evaluate gravity
 * (through N^2 interactions or by building the octree) every dt_g"): one evaluation a = accel(x_k), then
 * n_sub >= 1 semi-implicit Euler sub-steps of dt_c with that same a (dt_g = n_sub dt_c; contacts are out
 * of scope, so nothing else acts between evaluations).  Bit-identical to n_sub separate updates. */
bh_status bh_multirate_step(bh_ctx *ctx, double dt_c, int n_sub);

/* Gravitational potential of every body of the last build with the interaction lists of bh_accel
 * (same groups, same opening test):  phi_i = -G sum_k m_k / sqrt(|d|^2 + eps^2), a body skips itself, a
 * pair at zero softened distance adds nothing (R24: the potential whose gradient is the force of
 * Eqs. (4)-(6) PAPER.md:90-101; the paper checks energy conservation, but prints no
 * potential).  phi_dev is [n] in bh_build order.  Overwrites the counters read by bh_get_counts/stats. */
bh_status bh_potential(bh_ctx *ctx, double theta, double eps, double G, double *phi_dev);

/* Accelerations (as bh_accel) and potential (as bh_potential) of every body from ONE walk: the two share
 * the distance and the reciprocal square root of every interaction (19 fp64 instructions instead of 16 + 12),
 * so following the energy of a run costs a fifth more than the accelerations alone.
 * acc_dev [n][3], phi_dev [n], bh_build order. */
bh_status bh_accel_potential(bh_ctx *ctx, double theta, double eps, double G, double *acc_dev, double *phi_dev);

/* Direct-sum potential over all ordered pairs (the plain definition of the same phi). phi_dev [n]. */
bh_status bh_direct_potential(bh_ctx *ctx, double eps, double G, double *phi_dev);

/* Synchronising. Conserved quantities of n bodies given as device arrays:
 * out_host[0] = kinetic energy 1/2 sum m |v|^2;  [1] = potential energy 1/2 sum m_i phi_i (0 if phi_dev
 * is NULL);  [2..4] = linear momentum sum m v;  [5..7] = angular momentum sum m x cross v about the
 * origin.  Accumulated in double-double in a fixed order: reproducible run to run, and exact to fp64
 * rounding of the true sum of the fp64 inputs.  Needs no prior build. */
bh_status bh_diagnostics(bh_ctx *ctx, const double *pos_dev, const double *vel_dev, const double *mass_dev,
                         const double *phi_dev, int64_t n, double out_host[8]);

/* The same eight sums as bh_diagnostics, bit for bit, for callers that have no way to
 * allocate device memory: no context, no workspace, and no cudaMalloc / cudaFree or other allocating call inside.
 * That is the situation of code that is only ever handed device pointers: a plug-in or analysis hook inside
 * a host application whose memory pool owns the whole GPU (whatever such a hook allocated itself would come out
 * of nobody's budget and can fail once the pool has taken the card), a monitor called from inside a time-step
 * loop where cudaMalloc / cudaFree would stall every stream of the device, or a process under a fixed memory
 * quota.  Such a caller cannot provide the workspace bh_create asks for, so bh_diagnostics is out of its reach;
 * this call takes only the inputs, the output and a stream.
 *   pos_dev, vel_dev [n][3], mass_dev [n], phi_dev [n] or NULL: device arrays, read only.
 *   out_dev [8]: DEVICE array owned by the caller, receives ekin, epot, P[3], L[3] as in bh_diagnostics.
 *   cuda_stream: the cudaStream_t to enqueue on (NULL = legacy default stream).  The call does NOT wait for
 *   the GPU: read out_dev after synchronising the stream, or from later work on the same stream.
 * Scratch: the per-block partial sums and the ticket of the reduction sit in one array of
 * BH_DIAG_STATIC_SCRATCH_BYTES (76 032) bytes of device memory inside the library image; every GPU the process
 * uses with libbh loaded holds that much from load to exit, whether or not this call is ever made.  The array
 * is specified for n <= BH_DIAG_STATIC_MAX_N bodies (2^30, the most bodies any libbh call accepts); a larger n
 * is refused with BH_ERR_CAPACITY and a message naming both numbers.
 * First call on a device: looks up the device address of the array (cudaGetSymbolAddress, once per device, with
 * that device current) before it launches.  Make that first call outside any stream capture; later calls on the
 * same device only enqueue a 4-byte memset (the ticket) and the kernel.
 * Sharing: there is ONE array per GPU for the whole process and it keeps what the last call left in it.  Calls
 * that can run on the GPU at the same time (different streams, or different host threads without ordering
 * between their streams) overwrite each other's partial sums and both results are garbage: keep every use of
 * this call on one device in one stream order.  Calls on different GPUs do not interact.
 * Errors: BH_ERR_INVALID_ARG (null pointer other than phi_dev, n < 1), BH_ERR_CAPACITY (n too large),
 * BH_ERR_CUDA (address lookup, memset or launch failed); bh_last_error(NULL) returns the message (per host
 * thread).  Pointers are not checked for being device pointers. */
#define BH_DIAG_STATIC_MAX_N ((int64_t)1 << 30)
#define BH_DIAG_STATIC_SCRATCH_BYTES 76032
bh_status bh_diagnostics_static(const double *pos_dev, const double *vel_dev, const double *mass_dev,
                                const double *phi_dev, int64_t n, double *out_dev, void *cuda_stream);

/* Synchronising. Maximum relative position error in per cent, Eq. (7) PAPER.md:223:
 * max_i 100 |r_i - r_i,ref| / |r_i,ref|, with |.|^2 = fma(z,z,fma(y,y,x*x)), e_i = 100 sqrt(|d|^2/|r_ref|^2),
 * every operation IEEE-rounded once (bit-reproducible); bodies with r_ref at the origin are skipped (R25).
 * pos_dev, ref_dev are [n][3]. */
bh_status bh_position_error(bh_ctx *ctx, const double *pos_dev, const double *ref_dev, int64_t n,
                            double *err_host);

/* Synchronising. Broad phase of the collision detection over the bodies of the last
 * bh_build, on its octree: the bounding volume of body i is the sphere of radius
 * b_i = fma(|v_i|, dt, R_i) about its centre (R26: "estimated based on its velocity and integration time
 * step"; radius_dev [n] = circumscribed radius R_i, vel_dev [n][3] or NULL for b = R, both in bh_build
 * order); a pair i < j is reported iff |x_j - x_i|^2 <= (b_i + b_j)^2 (touching counts) with
 * d2 = fma(dz, dz, fma(dy, dy, dx*dx)) and every operation rounded once.  Pairs (i, j), i < j, are written
 * to pairs_dev [capacity][2] in no particular order, each once; *count_host = number found.  capacity 0
 * (pairs_dev may be NULL) only counts.  BH_ERR_CAPACITY if count > capacity > 0 (the first `capacity`
 * slots are filled, *count_host is valid: call again with a larger buffer). */
bh_status bh_broadphase(bh_ctx *ctx, const double *radius_dev, const double *vel_dev, double dt,
                        int32_t *pairs_dev, int64_t capacity, int64_t *count_host);

/* Synchronising. Aggregate identification: connected components of the graph whose
 * vertices are the n bodies and whose edges are the n_pairs contacts pairs_dev [n_pairs][2] (any order,
 * repeats and self-pairs allowed).  label_dev [n] = smallest body id of the body's component;
 * size_dev [n] (may be NULL) = number of bodies, at the component's label, 0 elsewhere; agg_mass_dev [n]
 * (may be NULL; needs mass_dev [n]) = total mass, same layout (atomic sums: order not fixed, ~n ulp).
 * counts_host[0] = components, [1] = aggregates = components with more than one body.
 * Needs no build; n <= max_n.  BH_ERR_INVALID_ARG if a pair names a body outside [0, n). */
bh_status bh_aggregates(bh_ctx *ctx, int64_t n, const int32_t *pairs_dev, int64_t n_pairs, const double *mass_dev,
                        int32_t *label_dev, int32_t *size_dev, double *agg_mass_dev, int64_t counts_host[2]);

/* Host helper. Upper bound of the gravity time step, Eq. (8): 1 / (2 sqrt(G rho)). */
double bh_gravity_dt(double G, double rho);

/* End-to-end evaluation from HOST buffers: copies pos_host [n][3] and mass_host [n] to the GPU,
 * builds, walks, delivers the accelerations in acc_host [n][3] and waits.  Pinned host memory makes the
 * copies asynchronous; pageable memory works too.  The masses travel on a second stream beside the first
 * build kernels (they are first needed after the sort).  If acc_host is pinned (cudaHostAlloc /
 * cudaHostRegister, e.g. a torch pin_memory() tensor) the walk kernel stores the accelerations straight into
 * it while it computes (the 24 bytes of a body in one store instruction of three adjacent lanes) and no copy
 * follows; otherwise they are staged in the workspace and copied.  Nothing else decides the path and no state
 * is carried between calls; both paths give the same bits. */
bh_status bh_eval_host(bh_ctx *ctx, const double *pos_host, const double *mass_host, int64_t n,
                       double theta, double eps, double G, double *acc_host);

/* Wait for the stream and report sticky errors (BH_ERR_NONFINITE, BH_ERR_CAPACITY, BH_ERR_CUDA). */
bh_status bh_synchronize(bh_ctx *ctx);

/* ---- inspection of the last build (parity tests, metrics) ---- */
/* Synchronising. Cube corner lo[3] and side L (a power of two, R11). */
bh_status bh_get_cube(bh_ctx *ctx, double lo_host[3], double *side_host);
/* Sorted keys [n] and the sort permutation perm [n] (sorted position -> bh_build index). */
bh_status bh_get_keys(bh_ctx *ctx, uint64_t *sorted_key_dev, uint32_t *perm_dev);
/* Synchronising. Node count M and depth (deepest level). */
bh_status bh_get_node_count(bh_ctx *ctx, int64_t *m_host, int32_t *depth_host);
/* Node arrays, each [M] (mono [M][4] = cx,cy,cz,m); any pointer may be NULL. Caller sizes them
 * with bh_get_node_count. */
bh_status bh_get_nodes(bh_ctx *ctx, uint8_t *level_dev, uint32_t *begin_dev, uint32_t *count_dev,
                       int32_t *first_child_dev, uint8_t *child_mask_dev, int32_t *parent_dev,
                       double *mono_dev);
/* Synchronising. Walk groups (R6): a group cell is a tree node with <= Gc bodies (or a
 * leaf) whose parent has more; each group cell is cut into runs of W consecutive sorted bodies;
 * groups are numbered in sorted-body order.  *ng_host = number of groups Ng; gstart_dev (may be
 * NULL, else room for Ng+1 <= n+1 entries) receives the first sorted body of each group, then n. */
bh_status bh_get_groups(bh_ctx *ctx, int64_t *ng_host, uint32_t *gstart_dev);
/* Synchronising. Sorted bodies [n][4] (x,y,z,m) and group boxes [Ng][3] each; any pointer may be NULL. */
bh_status bh_get_bodies(bh_ctx *ctx, double *sbody_dev, double *glo_dev, double *ghi_dev);
/* Synchronising. Per-group interaction-list lengths of the last bh_accel, each [Ng]. */
bh_status bh_get_counts(bh_ctx *ctx, uint32_t *n_mono_per_group_dev, uint32_t *n_direct_per_group_dev);

/* Synchronising. Totals of the last bh_accel: stats[0] = sum over groups of n_mono, stats[1] = sum
 * of n_direct, stats[2] = body-source interactions evaluated (sum of group bodies x list length),
 * stats[3] = nodes tested by the opening criterion, stats[4] = times a traversal stack outgrew shared
 * memory and spilled 128 entries to the workspace (deep or wide traversals: small theta). */
bh_status bh_get_stats(bh_ctx *ctx, uint64_t stats_host[BH_NUM_STATS]);

/* Number of CUDA kernels this context has launched since bh_create (memsets and copies excluded). */
bh_status bh_get_launches(bh_ctx *ctx, uint64_t *count_host);

/* Phase timing with CUDA events on the context's stream.  After bh_set_timing(ctx, 1) every
 * bh_build/bh_accel/bh_direct records events; bh_get_phase_ms (synchronising) returns the last
 * durations in ms: [0] cube, [1] keys+histogram, [2] sort, [3] gather+boxes, [4] tree,
 * [5] monopoles, [6] walk, [7] direct, [8] kick/drift kernels of the last bh_kdk_step.  A build of at most
 * 1024 bodies per multiprocessor is ONE kernel (one block up to 4096 bodies, one co-resident grid with grid
 * barriers above): its whole duration is reported as [4] and [0]-[3], [5] are 0.  A build reports only the phases
 * it ran itself: inside a bh_kdk_step above those sizes the drift kernel also takes the bounding cube of the
 * positions it writes, so [0] is 0 for that step's build and the cube's cost is part of [8]; a stepper that
 * evaluates gravity by the direct sum reports [7] and 0 for [0]-[6], one that walks the tree 0 for [7]. */
#define BH_NUM_PHASES 9
bh_status bh_set_timing(bh_ctx *ctx, int enable);
bh_status bh_get_phase_ms(bh_ctx *ctx, float ms_host[BH_NUM_PHASES]);

const char *bh_last_error(const bh_ctx *ctx);
const char *bh_version(void);

#ifdef __cplusplus
}
#endif
#endif /* BH_H_ */
