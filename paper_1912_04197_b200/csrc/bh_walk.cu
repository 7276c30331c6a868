// bh_walk.cu — step a7 (group-cooperative tree walk, Eqs. (3)-(6) PAPER.md:84-106), step a8 (direct
// N^2 sum, Eq. (1)) and step a9 (leapfrog kernels).
//
// Walk: a group is up to 32 Morton-consecutive bodies of one group cell (R6).  The kernel is warp
// specialised: one persistent 512-thread block per SM holds eight PAIRS of warps, a producer and a
// consumer, joined by a ring of sources (x,y,z,m) in shared memory.
//   producer  lanes = candidate nodes.  It takes a group from the atomic queue and traverses the tree
//             for it: pops up to 32 sibling ranges (first child, count) from a LIFO stack (shared-memory
//             ring, spill slab in global memory); every lane walks its range one node per trip and
//             applies the opening test of the GROUP (R3-R7: node edge s, distance from the node's
//             centre of mass to the group's bounding box, accept iff s*s < theta^2 d^2, never accept a
//             node that holds a body of the group); the results are appended by ballot/prefix:
//             accepted nodes -> their (cx,cy,cz,m) into the ring; opened internal nodes -> their child
//             range onto the stack; opened leaves -> their bodies (x,y,z,m) into the ring (cp.async,
//             straight from L2).  The record of a lane's next sibling is requested as soon as the accepted
//             monopoles of the trip are in the ring.  The producer is written for instruction count: on
//             sm_100 every integer / move / branch instruction another warp issues costs the fp64 warps of
//             the same sub-partition a dispatch cycle (loads, stores and shuffles do not).
//   consumer  lanes = bodies.  It evaluates the sources the producer has published, in fp64: every
//             lane carries FOUR bodies of the group (lane l: bodies l%8 + 8k) and the four quarter-warps
//             take alternate sources, so one shared-memory read of a source feeds four interactions and
//             the fp64 pipe, not the load-store path, sets the pace.  Sources are taken in blocks of 32
//             from a block-aligned ring position (bh_eval.cuh).
// The two roles meet only through release/acquire counters in shared memory, so the fp64 pipe of an SM
// sub-partition is fed by its two consumers while its two producers wait on L2.
// The test arithmetic is the canonical one (each operation rounded once, fma where stated) so that
// every accept/open decision equals the oracle's; traversal and accumulation order are free (R23).
#include "bh_eval.cuh"

namespace bh {

constexpr int kPairs = WalkConfig::kPairsPerBlock;       // producer/consumer pairs per block
constexpr int kWalkThreads = kPairs * 64;
constexpr int kStack = 512;                 // sibling ranges per producer in shared memory (ring)
constexpr int kSpill = 128;                 // spill / refill unit
constexpr int kDesc = 4;                    // group descriptors in flight per pair
constexpr unsigned kNoGroup = 0xffffffffu;
constexpr unsigned kSleepFullNs = 1000;     // ns a producer sleeps per poll while its ring is full
constexpr int kRegProd = 96;                // registers per thread of the producer warpgroups ...
constexpr int kRegCons = 160;               // ... and of the consumer warpgroups (launch: 128)
constexpr int kPubMin = 32;                 // a trip publishes only if more than this many entries are pending (the consumer starts a batch at 32)


constexpr int kMaxSplit = 4;                 // most consumer warps that share one producer's ring (see walk_kernel)

struct PairCtrl {                            // all words are written by one role and read by the other
    unsigned tail_pub;                       // producer: ring entries below this are complete
    unsigned started;                        // producer: groups whose descriptor is valid
    unsigned finished;                       // producer: groups whose list is complete (desc_end valid)
    unsigned head_pub[kMaxSplit];            // consumer s: ring entries below this are free again
    unsigned consumed[kMaxSplit];            // consumer s: groups it is done with
    unsigned desc_g[kDesc], desc_begin[kDesc], desc_end[kDesc];
    unsigned pad;
};

struct PairSmem {
    double4 ring[kRing];
    uint2 stack[kStack];                     // (first sibling, count) ranges
    unsigned leaf_src[2][32];                // producer scratch: (first body - offset in the run) per opened leaf, rows by trip parity
    PairCtrl ctrl;
};

struct WalkSmem {
    PairSmem pair[kPairs];
};

__device__ __forceinline__ void cp_async16(void *smem, const void *gmem)
{
    const unsigned s = (unsigned)__cvta_generic_to_shared(smem);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(s), "l"(gmem) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_1() { asm volatile("cp.async.wait_group 1;" ::: "memory"); }

__device__ __forceinline__ void st_release(unsigned *p, unsigned v)
{
    const unsigned a = (unsigned)__cvta_generic_to_shared(p);
    asm volatile("st.release.cta.shared.u32 [%0], %1;" ::"r"(a), "r"(v) : "memory");
}
__device__ __forceinline__ unsigned ld_acquire(const unsigned *p)
{
    const unsigned a = (unsigned)__cvta_generic_to_shared(p);
    unsigned v;
    asm volatile("ld.acquire.cta.shared.u32 %0, [%1];" : "=r"(v) : "r"(a) : "memory");
    return v;
}
// lane 0 reads a counter of the other role; the shuffle hands the value (and the ordering) to the warp
__device__ __forceinline__ unsigned warp_acquire(const unsigned *p, unsigned lane)
{
    unsigned v = 0;
    if (lane == 0) v = ld_acquire(p);
    return __shfl_sync(0xffffffffu, v, 0);
}
// the smallest of the first k counters of the other role (lanes < k read one each)
__device__ __forceinline__ unsigned warp_acquire_min(const unsigned *p, unsigned k, unsigned lane)
{
    unsigned v = 0xffffffffu;
    if (lane < k) v = ld_acquire(p + lane);
    return __reduce_min_sync(0xffffffffu, v);
}
// lane 0 publishes a counter after the whole warp has passed this point
__device__ __forceinline__ void warp_release(unsigned *p, unsigned v, unsigned lane)
{
    __syncwarp();
    if (lane == 0) st_release(p, v);
}

// ------------------------------------------------------------------------------------------ producer
struct Producer {
    PairSmem &ps;
    unsigned lane;
    unsigned tail;        // ring entries written (absolute)
    unsigned head_seen;   // smallest value last read from ctrl.head_pub[0 .. split)
    unsigned pub;         // last value stored to ctrl.tail_pub
    unsigned split;       // consumer warps that read this ring

    __device__ __forceinline__ void publish(unsigned v)
    {
        if ((int)(v - pub) > 0) {
            warp_release(&ps.ctrl.tail_pub, v, lane);
            pub = v;
        }
    }
    // make room for n more ring entries.  When the ring is full: publish everything written so far
    // (the consumer can only free what it has been given), then sleep until a good part of the ring
    // is free again, so that the producer works in bursts and does not burn issue slots polling
    __device__ __forceinline__ void reserve_slow(unsigned n)
    {
        cp_async_commit();
        cp_async_wait_all();
        publish(tail);
        const unsigned want = n > (unsigned)kRing / 2 - 64u ? n : (unsigned)kRing / 2 - 64u;
        while (true) {
            __nanosleep(kSleepFullNs);
            head_seen = warp_acquire_min(ps.ctrl.head_pub, split, lane);
            if (tail + want - head_seen <= (unsigned)kRing) break;
        }
    }
    __device__ __forceinline__ void reserve(unsigned n)
    {
        if (tail + n - head_seen <= (unsigned)kRing) return;
        head_seen = warp_acquire_min(ps.ctrl.head_pub, split, lane);
        if (tail + n - head_seen <= (unsigned)kRing) return;
        reserve_slow(n);
    }
};

struct NodeRec {
    uint4 info;      // begin, count, first_child, level | children << 8
    double4 mn;      // centre of mass, mass
};

__device__ __forceinline__ NodeRec load_rec(const uint4 *__restrict__ winfo, const double4 *__restrict__ mono, unsigned t)
{
    NodeRec r;
    r.info = __ldg(winfo + t);
    const double2 *m2 = reinterpret_cast<const double2 *>(mono + t);
    const double2 lo = __ldg(m2), hi = __ldg(m2 + 1);
    r.mn = make_double4(lo.x, lo.y, hi.x, hi.y);
    return r;
}

// max(0, max(lo - c, c - hi)), each difference rounded once (R22).  Since lo <= hi at most one of the
// differences is positive, so the result is picked on the integer pipe (an fp64 max costs six
// instructions on sm_100, and every instruction of a producer takes an issue slot from the fp64
// warps): high word = max(h1, h2, 0) as signed integers, low word = that of t1 if t1 >= 0, else of
// t2.  When neither difference is positive the high word is 0 and the low word arbitrary: a
// subnormal whose square rounds to zero, and the result is only ever squared (so is -0 for +0).
__device__ __forceinline__ double box_delta(double lo, double hi, double c)
{
    const double t1 = __dsub_rn(lo, c), t2 = __dsub_rn(c, hi);
    const int h1 = __double2hiint(t1), h2 = __double2hiint(t2);
    const int h = __vimax3_s32(h1, h2, 0);
    const int l = h1 >= 0 ? __double2loint(t1) : __double2loint(t2);
    return __hiloint2double(h, l);
}

// The stack holds RANGES of sibling nodes (first id, count): one entry per opened node.  A pop gives
// every lane one range; the lane then walks its (at most eight, memory-contiguous) siblings one per
// trip, so the warp-wide bookkeeping of a trip (two ballots, one stack entry per opened node) is
// spread over up to 32 nodes and the records of the next trip are already in flight.
// POT (potential walk): the group's own bodies enter the ring with zero mass; the consumer adds the
// pairs inside the group itself, where a body can be told from its coincident neighbours (R24).
template <bool POT>
__device__ void produce(PairSmem &ps, DevState *st, const unsigned *__restrict__ gstart,
                        const double4 *__restrict__ sbody, const double *__restrict__ gbox,
                        const uint4 *__restrict__ winfo, const double4 *__restrict__ mono, double theta2,
                        unsigned *__restrict__ cnt_mono, unsigned *__restrict__ cnt_direct, uint2 *slab, unsigned split)
{
    const unsigned lane = lane_id();
    const unsigned lt = (1u << lane) - 1u;
    const unsigned ngroups = st->n_groups;
    const int s2_base = (2 * st->e + 1023) << 20;   // high word of L^2; a level down is 2^-2: subtract 2 << 20 (|e| <= 301 is checked by cube_kernel, so the exponent field stays in range)
    unsigned long long tot_mono = 0, tot_direct = 0, tot_inter = 0, tot_tested = 0;
    unsigned tot_spills = 0;   // times the shared stack overflowed into the global slab (stats[4])
    Producer P{ps, lane, 0u, 0u, 0u, split};
    uint2 *stack = ps.stack;
    unsigned k = 0;   // groups started by this pair

    while (true) {
        unsigned g = 0;
        if (lane == 0) g = atomicAdd(&st->walk_queue, 1u);
        g = __shfl_sync(0xffffffffu, g, 0);
        if (g >= ngroups) g = kNoGroup;
        while (k - warp_acquire_min(ps.ctrl.consumed, split, lane) >= (unsigned)kDesc) __nanosleep(256);
        P.tail = (P.tail + 31u) & ~31u;        // a group's sources start on a block boundary (eval_blocks)
        if (lane == 0) {
            ps.ctrl.desc_g[k % kDesc] = g;
            ps.ctrl.desc_begin[k % kDesc] = P.tail;
        }
        warp_release(&ps.ctrl.started, k + 1, lane);
        if (g == kNoGroup) {
            // the last producer warp of the grid to run out of groups leaves the queue ready for the next walk
            if (lane == 0 && atomicAdd(&st->walk_done, 1u) == gridDim.x * ((unsigned)kPairs / split) - 1u) {
                st->walk_queue = 0u;
                st->walk_done = 0u;
            }
            break;
        }

        const unsigned gb = gstart[g], ge = gstart[g + 1];
        const double glx = gbox[6 * g + 0], gly = gbox[6 * g + 1], glz = gbox[6 * g + 2];
        const double ghx = gbox[6 * g + 3], ghy = gbox[6 * g + 4], ghz = gbox[6 * g + 5];
        unsigned bot = 0, top = 1, gsp = 0;    // shared stack = [bot, top) mod kStack; gsp entries in the slab
        unsigned n_direct = 0, n_tested = 0;
        const unsigned tail_begin = P.tail;    // the ring only ever receives this group's monopoles and bodies: n_mono follows from the tail
        if (lane == 0) stack[0] = make_uint2(0u, 1u);   // the root, as a range of one
        __syncwarp();
        unsigned tail_prev = P.tail;           // ring fill at the end of the previous trip

        while (true) {
            if (top == bot) {
                if (gsp == 0) break;           // nothing left: the list of this group is complete
                gsp -= kSpill;                 // refill from the slab
                for (unsigned q = lane; q < (unsigned)kSpill; q += 32) stack[(bot + q) & (kStack - 1)] = slab[gsp + q];
                top = bot + kSpill;
                __syncwarp();
            }
            unsigned take = top - bot;
            take = take < 32u ? take : 32u;
            top -= take;
            uint2 ent = make_uint2(0u, 0u);
            if (lane < take) ent = stack[(top + lane) & (kStack - 1)];
            __syncwarp();                      // the entries are read before later pushes reuse their slots
            const unsigned first = ent.x, nsib = ent.y;
            const unsigned trips = __reduce_max_sync(0xffffffffu, nsib);
            n_tested += __reduce_add_sync(0xffffffffu, nsib);   // every sibling of a popped range is tested
            // room for everything this pop can push (32 child ranges per trip): spill the oldest entries first
            while (top - bot + 32u * trips > (unsigned)kStack) {
                if (gsp + kSpill > (unsigned)kStackSlab) {      // cannot happen within the slab bound
                    if (lane == 0) atomicOr(&st->status, (int)kStatStack);
                    bot = top;                                  // drop the stack: the walk ends early
                } else {
                    for (unsigned u = lane; u < (unsigned)kSpill; u += 32) slab[gsp + u] = stack[(bot + u) & (kStack - 1)];
                    gsp += kSpill;
                    bot += kSpill;
                    ++tot_spills;
                }
            }
            NodeRec nxt;
            nxt.info = make_uint4(0u, 0u, 0u, 0u);
            nxt.mn = make_double4(0.0, 0.0, 0.0, 0.0);
            if (nsib > 0) nxt = load_rec(winfo, mono, first);
#pragma unroll 1
            for (unsigned q = 0; q < trips; ++q) {
                const bool have = q < nsib;
                const NodeRec cur = nxt;
                // ---- opening test (canonical arithmetic, R22) ----
                const unsigned nb = cur.info.x, nc = cur.info.y;
                const bool internal = (int)cur.info.z >= 0;
                const bool overlap = (nb < ge) && (gb < nb + nc);
                const double dx = box_delta(glx, ghx, cur.mn.x);
                const double dy = box_delta(gly, ghy, cur.mn.y);
                const double dz = box_delta(glz, ghz, cur.mn.z);
                const double d2 = __fma_rn(dz, dz, __fma_rn(dy, dy, __dmul_rn(dx, dx)));
                const double s2 = __hiloint2double(s2_base - (int)((cur.info.w & 0xffu) << 21), 0);   // (L 2^-level)^2
                const bool accept = have && !overlap && (s2 < __dmul_rn(theta2, d2));
                const bool open_int = have && !accept && internal;
                const bool open_leaf = have && !accept && !internal;
                // the three votes side by side: ptxas guards every warp collective that follows a branch with a
                // convergence check (two instructions), and adjacent ones share it
                const unsigned m_acc = __ballot_sync(0xffffffffu, accept);
                const unsigned m_int = __ballot_sync(0xffffffffu, open_int);
                const unsigned m_leaf = __ballot_sync(0xffffffffu, open_leaf);
                // ---- accepted nodes -> ring ----
                {
                    const unsigned m = m_acc;
                    const unsigned cnt = __popc(m);
                    P.reserve(cnt);
                    if (accept) ps.ring[(P.tail + __popc(m & lt)) & (kRing - 1)] = cur.mn;
                    P.tail += cnt;
                }
                // the record of the lane's next sibling is requested once the accepted monopoles are in the ring: the
                // centre-of-mass registers are free by then, so only the four info words have to be kept aside
                // (requested at the top of the trip the whole record is copied every trip: 5.09 -> 5.05 ms)
                const unsigned fc = cur.info.z, lw = cur.info.w;
                if (q + 1 < nsib) nxt = load_rec(winfo, mono, first + q + 1);
                // ---- opened internal nodes -> their child ranges onto the stack ----
                {
                    const unsigned m = m_int;
                    if (m) {
                        // slot and value computed by every lane, only the store is predicated (no branch around it)
                        const unsigned slot = (top + __popc(m & lt)) & (kStack - 1);
                        const uint2 range = make_uint2(fc, (lw >> 8) & 0xffu);
                        if (open_int) stack[slot] = range;
                        top += __popc(m);
                    }
                }
                // ---- opened leaves -> their bodies, asynchronously into the ring ----
                // All opened leaves of the trip are expanded together: a warp scan gives every leaf its
                // offset in the run of bodies, the leaves leave (first body - offset) in a scratch row,
                // and every lane then copies one body per window of 32, finding its leaf by counting
                // the leaf starts at or before its slot.
                {
                    const unsigned m = m_leaf;
                    if (m) {
                        const unsigned c = open_leaf ? nc : 0u;
                        unsigned inc = c;
#pragma unroll
                        for (int o = 1; o < 32; o <<= 1) {
                            const unsigned t = __shfl_up_sync(0xffffffffu, inc, o);
                            if (lane >= (unsigned)o) inc += t;
                        }
                        const unsigned total = __shfl_sync(0xffffffffu, inc, 31);
                        const unsigned excl = inc - c;
                        unsigned *lsrc = ps.leaf_src[q & 1u];          // alternate rows: the next trip does not wait for this one's reads
                        if (open_leaf) lsrc[__popc(m & lt)] = nb - excl;
                        __syncwarp();
                        unsigned owners = 0;                           // leaves that start before this window
                        for (unsigned base = 0; base < total; base += 32) {
                            const unsigned rel = excl - base;
                            const unsigned heads = __reduce_or_sync(0xffffffffu, (open_leaf && rel < 32u) ? 1u << rel : 0u);
                            const unsigned k = owners + __popc(heads & (lt | (1u << lane))) - 1u;
                            owners += __popc(heads);
                            const unsigned n = total - base < 32u ? total - base : 32u;
                            P.reserve(n);
                            if (lane < n) {
                                char *dst = reinterpret_cast<char *>(&ps.ring[(P.tail + lane) & (kRing - 1)]);
                                const unsigned src = lsrc[k] + base + lane;
                                const char *from = reinterpret_cast<const char *>(sbody + src);
                                if (POT && src >= gb && src < ge) {
                                    ps.ring[(P.tail + lane) & (kRing - 1)] = make_double4(0.0, 0.0, 0.0, 0.0);
                                } else {
                                    cp_async16(dst, from);
                                    cp_async16(dst + 16, from + 16);
                                }
                            }
                            P.tail += n;
                        }
                        n_direct += total;
                    }
                }
                // ---- publish what is complete: everything up to the end of the previous trip ----
                cp_async_commit();
                if ((int)(tail_prev - P.pub) > kPubMin) {
                    cp_async_wait_1();
                    P.publish(tail_prev);
                }
                tail_prev = P.tail;
            }
            __syncwarp();                      // this batch's pushes are on the stack before the next pop
        }
        // ---- the list of this group is complete ----
        cp_async_wait_all();
        __syncwarp();
        const unsigned n_mono = P.tail - tail_begin - n_direct;
        if (lane == 0) {
            ps.ctrl.desc_end[k % kDesc] = P.tail;
            st_release(&ps.ctrl.tail_pub, P.tail);
            st_release(&ps.ctrl.finished, k + 1);
            cnt_mono[g] = n_mono;
            cnt_direct[g] = n_direct;
        }
        P.pub = P.tail;
        ++k;
        tot_mono += n_mono;
        tot_direct += n_direct;
        tot_inter += (unsigned long long)(n_mono + n_direct) * (unsigned long long)(ge - gb);
        tot_tested += n_tested;                // warp-uniform
    }
    if (lane == 0) {
        atomicAdd(&st->stats[0], tot_mono);
        atomicAdd(&st->stats[1], tot_direct);
        atomicAdd(&st->stats[2], tot_inter);
        atomicAdd(&st->stats[3], tot_tested);
        if (tot_spills) atomicAdd(&st->stats[4], (unsigned long long)tot_spills);
    }
}

// ------------------------------------------------------------------------------------------ consumer
// A consumer that holds none of the group's bodies (split walk, group of fewer bodies than consumers): it only
// follows the producer so that the ring space it is counted for is released.
__device__ __forceinline__ void drain_group(PairSmem &ps, unsigned k, unsigned sub)
{
    const unsigned lane = lane_id();
    while (true) {
        unsigned lim = 0;
        bool fin = false;
        if (lane == 0) {
            const unsigned tp = ld_acquire(&ps.ctrl.tail_pub);      // tail_pub first, then finished (see consume_group)
            fin = (int)(ld_acquire(&ps.ctrl.finished) - k) > 0;
            lim = fin ? ps.ctrl.desc_end[k % kDesc] : tp;
            if (fin || (int)(lim - ps.ctrl.desc_begin[k % kDesc]) > 0) st_release(&ps.ctrl.head_pub[sub], lim);
        }
        if (__shfl_sync(0xffffffffu, (int)fin, 0)) break;
        __nanosleep(256);
    }
}

// one group: evaluate its sources as the producer publishes them, then write the accelerations.
// This consumer holds NS slots of eight bodies: slots sub, sub + split, ... of the group (split = 1: all of them).
template <bool GUARD, int NS, int MODE>
__device__ __forceinline__ void consume_group(PairSmem &ps, unsigned k, unsigned head, long long gb, long long ge,
                                              const double4 *__restrict__ sbody, const unsigned *__restrict__ perm,
                                              double eps2, double G, double *__restrict__ acc, double *__restrict__ phi,
                                              unsigned sub, unsigned split)
{
    const unsigned lane = lane_id(), quarter = lane >> 3, r = lane & 7u;
    Bodies<NS> B;
#pragma unroll
    for (int s = 0; s < NS; ++s) {
        const long long j = gb + r + 8 * (sub + s * split);
        const double4 bd = sbody[j < ge ? j : gb];
        B.x[s] = bd.x; B.y[s] = bd.y; B.z[s] = bd.z;
        B.ax[s] = B.ay[s] = B.az[s] = B.ph[s] = 0.0;
    }
    const double4 zero4 = make_double4(0.0, 0.0, 0.0, 0.0);
    while (true) {
        unsigned lim = 0;
        bool fin = false;
        if (lane == 0) {
            // tail_pub FIRST, then finished: if the group is not finished at the second load, the earlier
            // tail_pub cannot yet include entries of a later group (the producer publishes those only after
            // it has finished this one)
            const unsigned tp = ld_acquire(&ps.ctrl.tail_pub);
            fin = (int)(ld_acquire(&ps.ctrl.finished) - k) > 0;
            lim = fin ? ps.ctrl.desc_end[k % kDesc] : tp;
        }
        fin = __shfl_sync(0xffffffffu, (int)fin, 0) != 0;
        lim = __shfl_sync(0xffffffffu, lim, 0);
        const int avail = (int)(lim - head);       // negative while tail_pub still belongs to the last group
        if (!fin && avail < 32) {
            __nanosleep(32);
            continue;
        }
        // whole blocks of 32 sources (the group's list starts on a multiple of 32 in the ring, so head stays one
        // until the list ends); the chunks of eight that are left once the list is complete
        const unsigned n32 = avail > 0 ? ((unsigned)avail & ~31u) : 0u;
        eval_blocks<GUARD, NS, MODE>(ps.ring, head, n32, quarter, eps2, B);
        head += n32;
        if (fin) {
            const unsigned n8 = (unsigned)(avail > 0 ? avail : 0) & 24u;
            eval_chunks<GUARD, NS, MODE>(ps.ring, head, n8, quarter, eps2, B);
            head += n8;
            const unsigned rest = (unsigned)(avail > 0 ? avail : 0) & 7u;
            if (rest) {                             // last, partial chunk: absent sources are massless
                const double4 *p = ps.ring + (head & (kRing - 1)) + quarter;
                const double4 s0 = quarter < rest ? p[0] : zero4;
                const double4 s1 = quarter + 4 < rest ? p[4] : zero4;
#pragma unroll
                for (int s = 0; s < NS; ++s) interact_any<GUARD, MODE>(B.x[s], B.y[s], B.z[s], eps2, s0, B.ax[s], B.ay[s], B.az[s], B.ph[s]);
#pragma unroll
                for (int s = 0; s < NS; ++s) interact_any<GUARD, MODE>(B.x[s], B.y[s], B.z[s], eps2, s1, B.ax[s], B.ay[s], B.az[s], B.ph[s]);
                head += rest;
            }
            warp_release(&ps.ctrl.head_pub[sub], head, lane);
            break;
        }
        warp_release(&ps.ctrl.head_pub[sub], head, lane);
    }
    if constexpr (MODE != 0) {
        // pairs inside the group: quarter q takes the group's bodies gb + q, gb + q + 4, ...; a body skips itself
        for (long long k = gb + quarter; k < ge; k += 4) {
            const double4 sk = sbody[k];
#pragma unroll
            for (int s = 0; s < NS; ++s) {
                double4 src = sk;
                if (k == gb + r + 8 * (sub + s * split)) src.w = 0.0;
                interact_any<true, MODE>(B.x[s], B.y[s], B.z[s], eps2, src, B.ax[s], B.ay[s], B.az[s], B.ph[s]);
            }
        }
    }
    // add the four quarter-warp partial sums; lane 8 q + r then writes the body of slot q: r + 8 (sub + q split)
    double ox = 0.0, oy = 0.0, oz = 0.0, op = 0.0;
#pragma unroll
    for (int s = 0; s < NS; ++s) {
        if constexpr (MODE == 2) {
            double tp = B.ph[s];
            tp += __shfl_xor_sync(0xffffffffu, tp, 8);
            tp += __shfl_xor_sync(0xffffffffu, tp, 16);
            if ((int)quarter == s) op = tp;
        }
        double tx = B.ax[s], ty = B.ay[s], tz = B.az[s];
        tx += __shfl_xor_sync(0xffffffffu, tx, 8);
        ty += __shfl_xor_sync(0xffffffffu, ty, 8);
        tz += __shfl_xor_sync(0xffffffffu, tz, 8);
        tx += __shfl_xor_sync(0xffffffffu, tx, 16);
        ty += __shfl_xor_sync(0xffffffffu, ty, 16);
        tz += __shfl_xor_sync(0xffffffffu, tz, 16);
        if ((int)quarter == s) { ox = tx; oy = ty; oz = tz; }
    }
    const long long j = gb + r + 8 * (sub + quarter * split);
    const bool mine = (int)quarter < NS && j < ge;
    const unsigned i = mine ? perm[j] : 0xffffffffu;
    if constexpr (MODE == 1) {
        if (mine) acc[i] = -G * ox;                 // phi, one value per body
    } else {
        if constexpr (MODE == 2) {
            if (mine) phi[i] = -G * op;
        }
        // The three components of a body go out in ONE store instruction from three adjacent lanes (value
        // v = 32 k + lane of instruction k is component v % 3 of the body held by lane v / 3), so the 24 bytes of a
        // body leave as one or two write segments instead of three: it matters when acc is pinned host memory
        // (bh_eval_host) and every segment is a PCIe write.
        const double a0 = G * ox, a1 = G * oy, a2 = G * oz;
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            const unsigned v = 32u * k + lane, src = v / 3u, c = v - 3u * src;
            const unsigned is = __shfl_sync(0xffffffffu, i, src);
            const double b0 = __shfl_sync(0xffffffffu, a0, src), b1 = __shfl_sync(0xffffffffu, a1, src),
                         b2 = __shfl_sync(0xffffffffu, a2, src);
            if (is != 0xffffffffu) acc[3ll * is + c] = c == 0u ? b0 : (c == 1u ? b1 : b2);
        }
    }
}

template <bool GUARD, int MODE>
__device__ void consume(PairSmem &ps, const unsigned *__restrict__ gstart, const double4 *__restrict__ sbody,
                        const unsigned *__restrict__ perm, double eps2, double G, double *__restrict__ acc,
                        double *__restrict__ phi, unsigned sub, unsigned split)
{
    const unsigned lane = lane_id();
    for (unsigned k = 0;; ++k) {
        while ((int)(warp_acquire(&ps.ctrl.started, lane) - k) <= 0) __nanosleep(64);
        const unsigned g = ps.ctrl.desc_g[k % kDesc];
        if (g == kNoGroup) break;
        const unsigned head = ps.ctrl.desc_begin[k % kDesc];
        const long long gb = gstart[g];
        const long long ge = gstart[g + 1];
        const int all = (int)((ge - gb + 7) >> 3);                                    // slots of eight bodies in the group
        const int slots = all > (int)sub ? (all - (int)sub + (int)split - 1) / (int)split : 0;   // ... that are mine
        if (slots >= 4) consume_group<GUARD, 4, MODE>(ps, k, head, gb, ge, sbody, perm, eps2, G, acc, phi, sub, split);
        else if (slots == 3) consume_group<GUARD, 3, MODE>(ps, k, head, gb, ge, sbody, perm, eps2, G, acc, phi, sub, split);
        else if (slots == 2) consume_group<GUARD, 2, MODE>(ps, k, head, gb, ge, sbody, perm, eps2, G, acc, phi, sub, split);
        else if (slots == 1) consume_group<GUARD, 1, MODE>(ps, k, head, gb, ge, sbody, perm, eps2, G, acc, phi, sub, split);
        else drain_group(ps, k, sub);
        warp_release(&ps.ctrl.consumed[sub], k + 1, lane);
    }
}

template <bool GUARD, int MODE>
__global__ void __launch_bounds__(kWalkThreads, 1)
walk_kernel(DevState *st, const unsigned *__restrict__ gstart, const double4 *__restrict__ sbody,
            const double *__restrict__ gbox, const unsigned *__restrict__ perm,
            const uint4 *__restrict__ winfo, const double4 *__restrict__ mono, double theta2, double eps2,
            double G, double *__restrict__ acc, unsigned *__restrict__ cnt_mono,
            unsigned *__restrict__ cnt_direct, unsigned *walk_stack, double *__restrict__ phi)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    WalkSmem &sm = *reinterpret_cast<WalkSmem *>(smem_raw);
    // warps 0-3 and 8-11 produce, 4-7 and 12-15 consume: every SM sub-partition (warp % 4) gets two of each
    const unsigned warp = threadIdx.x >> 5;
    const unsigned pair = (warp >> 3) * 4 + (warp & 3u);
    const bool producer = ((warp >> 2) & 1u) == 0;
    // Few groups (fewer than half / a quarter of the grid's consumer warps: configs[0], configs[1], PAPER.md:199's
    // N <= 10^4): `split` = 2 or 4 consumer warps share the ring of ONE producer and divide the group's BODIES
    // among them (slots of eight: consumer s takes slots s, s + split, ...), so a group's evaluation takes a
    // half / a quarter of the time and all fp64 pipes stay busy.  Every body still meets every source in the
    // same order: the results are bit-identical to the unsplit walk.  Pairs p with p % split == 0 lead; the
    // other producers have nothing to do.
    const unsigned ngroups = st->n_groups;
    const unsigned split = ngroups <= gridDim.x * (unsigned)kPairs / 4u ? 4u : (ngroups <= gridDim.x * (unsigned)kPairs / 2u ? 2u : 1u);
    const unsigned sub = pair % split;
    PairSmem &ps = sm.pair[pair - sub];
    if (producer && sub == 0 && lane_id() < sizeof(PairCtrl) / 4) reinterpret_cast<unsigned *>(&ps.ctrl)[lane_id()] = 0u;
    __syncthreads();
    // the block is launched with 128 registers per thread; the producer warpgroups hand registers to
    // the consumer warpgroups (warps 0-3 / 4-7 / 8-11 / 12-15 are the four warpgroups)
    if (producer) asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(kRegProd));
    else asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(kRegCons));
    if (producer) {
        if (sub == 0)
            produce<MODE != 0>(ps, st, gstart, sbody, gbox, winfo, mono, theta2, cnt_mono, cnt_direct,
                    reinterpret_cast<uint2 *>(walk_stack) + (size_t)(blockIdx.x * kPairs + pair) * kStackSlab, split);
    } else {
        consume<GUARD, MODE>(ps, gstart, sbody, perm, eps2, G, acc, phi, sub, split);
    }
}

// ------------------------------------------------------------------------------------------ a8
// Direct sum: two targets per thread (each source read from shared memory serves two interactions),
// sources streamed through 256-body shared-memory tiles.  When there are few targets the source range
// is split over blockIdx.y so that every SM has work; the partial sums are then added in split order
// by direct_reduce_kernel (deterministic).
constexpr int kDirectThreads = 256;
// kDirectPer targets per thread: one shared-memory read of a source feeds that many interactions.  Four when
// there are targets enough to fill the machine that way (1.026e12 against 1.009e12 interactions/s at N = 1M),
// two for smaller sets, where the number of blocks matters more (N = 16384: 1.9 against 2.7 ms).
template <bool GUARD, bool POT, int kDirectPer>
__global__ void __launch_bounds__(kDirectThreads, 2)
direct_kernel(long long n, const double4 *__restrict__ sbody, const unsigned *__restrict__ perm,
              const unsigned *__restrict__ iperm, const int32_t *__restrict__ tgt, long long nt, double eps2,
              double G, double *__restrict__ acc, double *__restrict__ partial, int tiles_per_split)
{
    constexpr int kDirectTargets = kDirectPer * kDirectThreads;
    __shared__ double4 tile[kDirectThreads];
    // all bodies: row r is sorted body r, written to its original index; sampled: row r is target tgt[r]
    long long r[kDirectPer], j[kDirectPer];
    double px[kDirectPer], py[kDirectPer], pz[kDirectPer], ax[kDirectPer], ay[kDirectPer], az[kDirectPer];
#pragma unroll
    for (int t = 0; t < kDirectPer; ++t) {
        r[t] = (long long)blockIdx.x * kDirectTargets + t * kDirectThreads + threadIdx.x;
        j[t] = r[t] < nt ? (tgt ? (long long)iperm[tgt[r[t]]] : r[t]) : 0;
        const double4 p = sbody[j[t]];
        px[t] = p.x; py[t] = p.y; pz[t] = p.z;
        ax[t] = ay[t] = az[t] = 0.0;
    }
    const long long s_begin = (long long)blockIdx.y * tiles_per_split * kDirectThreads;
    long long s_end = s_begin + (long long)tiles_per_split * kDirectThreads;
    if (s_end > n) s_end = n;
    for (long long t0 = s_begin; t0 < s_end; t0 += kDirectThreads) {
        const long long k = t0 + threadIdx.x;
        tile[threadIdx.x] = k < s_end ? sbody[k] : make_double4(0.0, 0.0, 0.0, 0.0);   // zero mass: no pull
        __syncthreads();
#pragma unroll 4
        for (int q = 0; q < kDirectThreads; ++q) {
            const double4 sq = tile[q];
#pragma unroll
            for (int t = 0; t < kDirectPer; ++t) {
                if constexpr (POT) {             // a body skips itself: its own term m/eps is not zero
                    double4 st = sq;
                    if (t0 + q == j[t]) st.w = 0.0;
                    interact_pot<GUARD>(px[t], py[t], pz[t], eps2, st, ax[t]);
                } else {
                    interact<GUARD>(px[t], py[t], pz[t], eps2, sq, ax[t], ay[t], az[t]);
                }
            }
        }
        __syncthreads();
    }
#pragma unroll
    for (int t = 0; t < kDirectPer; ++t) {
        if (r[t] >= nt) continue;
        if constexpr (POT) {                 // one value per body: phi = -G sum m / r
            if (gridDim.y == 1) acc[tgt ? r[t] : (long long)perm[r[t]]] = -G * ax[t];
            else partial[(size_t)blockIdx.y * nt + r[t]] = ax[t];
        } else if (gridDim.y == 1) {
            const long long o = tgt ? r[t] : (long long)perm[r[t]];
            acc[3 * o + 0] = G * ax[t]; acc[3 * o + 1] = G * ay[t]; acc[3 * o + 2] = G * az[t];
        } else {
            double *p = partial + (size_t)blockIdx.y * nt * 3;
            p[3 * r[t] + 0] = ax[t]; p[3 * r[t] + 1] = ay[t]; p[3 * r[t] + 2] = az[t];
        }
    }
}

// ncomp = 3 (accelerations, scale G) or 1 (potential, scale -G)
__global__ void direct_reduce_kernel(const double *__restrict__ partial, long long nt, int splits, double scale,
                                     int ncomp, const unsigned *__restrict__ perm, bool sampled,
                                     double *__restrict__ acc)
{
    for (long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x; k < ncomp * nt;
         k += (long long)gridDim.x * blockDim.x) {
        double s = 0.0;
        for (int q = 0; q < splits; ++q) s += partial[(size_t)q * nt * ncomp + k];
        const long long r = k / ncomp, c = k - ncomp * r;
        const long long o = sampled ? r : (long long)perm[r];
        acc[ncomp * o + c] = scale * s;
    }
}

// ------------------------------------------------------------------------------------------ a9
__global__ void kick_drift_kernel(double *__restrict__ pos, double *__restrict__ vel, const double *__restrict__ acc,
                                  long long n3, double h, double dt)
{
    for (long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x; k < n3;
         k += (long long)gridDim.x * blockDim.x) {
        const double v = __fma_rn(acc[k], h, vel[k]);
        vel[k] = v;
        pos[k] = __fma_rn(v, dt, pos[k]);
    }
}

__global__ void kick_kernel(double *__restrict__ vel, const double *__restrict__ acc, long long n3, double h)
{
    for (long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x; k < n3;
         k += (long long)gridDim.x * blockDim.x)
        vel[k] = __fma_rn(acc[k], h, vel[k]);
}

// ------------------------------------------------------------------------------------------ launchers
template <bool GUARD, int MODE>
static void launch_walk_t(const Workspace &w, double theta, double eps2, double G, double *out, double *phi, cudaStream_t s)
{
    static std::atomic<bool> configured[kMaxDevices];   // the attribute is per device
    const int dev = current_device();
    if (!configured[dev].load(std::memory_order_relaxed)) {
        cudaFuncSetAttribute(walk_kernel<GUARD, MODE>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(WalkSmem));
        configured[dev].store(true, std::memory_order_relaxed);
    }
    const int blocks = w.walk_warps / kPairs;   // one persistent block per SM
    walk_kernel<GUARD, MODE><<<blocks, kWalkThreads, sizeof(WalkSmem), s>>>(
        w.st, w.gstart, w.sbody, w.gbox, w.idx[0], w.winfo, w.mono, theta * theta, eps2, G, out, w.cnt_mono,
        w.cnt_direct, w.walk_stack, phi);
}

void launch_walk(const Workspace &w, int64_t n, double theta, double eps, double G, double *acc, int mode, double *phi,
                 cudaStream_t s)
{
    (void)n;
    const double eps2 = eps * eps;
    const bool guard = !(eps2 >= kTinyR2);
    if (mode == 1) {
        if (guard) launch_walk_t<true, 1>(w, theta, eps2, G, acc, nullptr, s);
        else launch_walk_t<false, 1>(w, theta, eps2, G, acc, nullptr, s);
    } else if (mode == 2) {
        if (guard) launch_walk_t<true, 2>(w, theta, eps2, G, acc, phi, s);
        else launch_walk_t<false, 2>(w, theta, eps2, G, acc, phi, s);
    } else {
        if (guard) launch_walk_t<true, 0>(w, theta, eps2, G, acc, nullptr, s);
        else launch_walk_t<false, 0>(w, theta, eps2, G, acc, nullptr, s);
    }
}

int launch_direct(const Workspace &w, int64_t n, const int32_t *tgt, int64_t nt, double eps, double G,
                  double *acc, bool potential, cudaStream_t s)
{
    const int64_t rows = tgt ? nt : n;
    const int per = rows >= 262144 ? 4 : 2;
    const int tblocks = (int)((rows + per * kDirectThreads - 1) / (per * kDirectThreads));
    const int tiles = (int)((n + kDirectThreads - 1) / kDirectThreads);
    // enough blocks for ~8 per SM; the partial sums live in the host-staging area (3 * max_n doubles)
    int splits = (w.sms * 8 + tblocks - 1) / tblocks;
    if (splits > tiles) splits = tiles;
    const int64_t room = w.stage_doubles / (3 * rows);
    if (splits > room) splits = (int)room;
    if (splits < 1) splits = 1;
    const int tps = (tiles + splits - 1) / splits;
    splits = (tiles + tps - 1) / tps;
    const double eps2 = eps * eps;
    dim3 grid(tblocks, splits);
    if (tgt) launch_iperm(w, n, s);   // sampled targets are named by body index: sorted position = iperm[index]
#define BH_DIRECT(GUARD, POT)                                                                                          \
    do {                                                                                                               \
        if (per == 4)                                                                                                  \
            direct_kernel<GUARD, POT, 4><<<grid, kDirectThreads, 0, s>>>(n, w.sbody, w.idx[0], w.iperm, tgt, rows,     \
                                                                         eps2, G, acc, w.stage_pos, tps);              \
        else                                                                                                           \
            direct_kernel<GUARD, POT, 2><<<grid, kDirectThreads, 0, s>>>(n, w.sbody, w.idx[0], w.iperm, tgt, rows,     \
                                                                         eps2, G, acc, w.stage_pos, tps);              \
    } while (0)
    if (potential) {
        if (eps2 >= kTinyR2) BH_DIRECT(false, true);
        else BH_DIRECT(true, true);
    } else {
        if (eps2 >= kTinyR2) BH_DIRECT(false, false);
        else BH_DIRECT(true, false);
    }
#undef BH_DIRECT
    if (splits > 1)
        direct_reduce_kernel<<<w.sms * 2, 256, 0, s>>>(w.stage_pos, rows, splits, potential ? -G : G,
                                                     potential ? 1 : 3, w.idx[0], tgt != nullptr, acc);
    return (splits > 1 ? 2 : 1) + (tgt ? 1 : 0);
}

void launch_kick_drift(double *pos, double *vel, const double *acc, int64_t n, double dt, cudaStream_t s)
{
    const long long n3 = 3ll * n;
    int blocks = (int)((n3 + 1023) / 1024);
    if (blocks > sm_count() * 8) blocks = sm_count() * 8;
    kick_drift_kernel<<<blocks, 256, 0, s>>>(pos, vel, acc, n3, dt * 0.5, dt);
}

void launch_kick(double *vel, const double *acc, int64_t n, double h, cudaStream_t s)
{
    const long long n3 = 3ll * n;
    int blocks = (int)((n3 + 1023) / 1024);
    if (blocks > sm_count() * 8) blocks = sm_count() * 8;
    kick_kernel<<<blocks, 256, 0, s>>>(vel, acc, n3, h);
}

}  // namespace bh
