// bh_contact.cu — rows NEXT-3 and NEXT-4 of SURVEY.md §8(f).
//
// NEXT-3  Broad phase of the collision detection: "pairs of bodies whose geometrical
//   boundaries are close enough are identified.  The bounding volume of a body is estimated based on its
//   velocity and integration time step."  Reading R26: bounding sphere of radius b_i = fma(|v_i|, dt, R_i);
//   a pair is a candidate iff d2 <= (b_i + b_j)^2 with d2 = fma(dz, dz, fma(dy, dy, dx*dx)), every
//   operation rounded once (the set of pairs is reproducible bit for bit).  The search reuses the octree
//   of the gravity step (rows a1-a5): an upward pass gives every node the exact box of its bodies'
//   centres and their largest b; a warp takes a walk group (<= 32 Morton-neighbours), descends from the
//   root with lanes = nodes, prunes a node iff its box is farther from the group's box than the two
//   largest radii allow, and tests the bodies of the surviving leaves against its own bodies (lanes =
//   bodies).  The pruning test uses the same, monotone, arithmetic as the pair test (box gaps <= true
//   gaps, radii >= true radii), so it can never drop a pair the exact rule accepts.  Every pair is found
//   once: from the body that comes first in the sorted order.
// NEXT-4  Aggregate identification: connected components of the contact graph (the
//   paper walks it by depth-first search, O(N+E)); here a lock-free union-find: every pair hooks the
//   larger root under the smaller (atomicCAS), so the root of a component is its smallest body id — the
//   canonical label — then one flattening pass, sizes and masses by atomics.
#include "bh_common.cuh"

namespace bh {

// ------------------------------------------------------------------------------------------ NEXT-3
__global__ void __launch_bounds__(256) bound_radius_kernel(const double *__restrict__ radius,
                                                           const double *__restrict__ vel,
                                                           const unsigned *__restrict__ perm, long long n, double dt,
                                                           double *__restrict__ bsort)
{
    const long long j = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= n) return;
    const unsigned i = perm[j];
    double b = radius[i];
    if (vel) {
        const double vx = vel[3ll * i], vy = vel[3ll * i + 1], vz = vel[3ll * i + 2];
        const double sp = __dsqrt_rn(__fma_rn(vz, vz, __fma_rn(vy, vy, __dmul_rn(vx, vx))));
        b = __fma_rn(sp, dt, b);
    }
    bsort[j] = b;
}

__device__ __forceinline__ double4 ldcg_d4(const double4 *p)
{
    const double2 *q = reinterpret_cast<const double2 *>(p);
    const double2 a = __ldcg(q), b = __ldcg(q + 1);
    return make_double4(a.x, a.y, b.x, b.y);
}

// box_lo[t] = (min x, min y, min z, max b), box_hi[t] = (max x, max y, max z, 0) over the bodies of node t.
// Leaves from their bodies; the last child to arrive (counter cnt[parent]) combines the children.
__global__ void __launch_bounds__(256) node_box_kernel(const DevState *__restrict__ st,
                                                       const double4 *__restrict__ sbody,
                                                       const double *__restrict__ bsort,
                                                       const uint4 *__restrict__ winfo,
                                                       const int *__restrict__ nparent, unsigned *cnt,
                                                       double4 *box_lo, double4 *box_hi, long long node_cap)
{
    const int M = st->n_nodes;
    if ((long long)M > node_cap) return;
    for (int t = blockIdx.x * blockDim.x + threadIdx.x; t < M; t += gridDim.x * blockDim.x) {
        const uint4 info = winfo[t];
        if ((int)info.z >= 0) continue;   // internal nodes are made by their last child
        double4 lo = sbody[info.x];
        double4 hi = lo;
        lo.w = bsort[info.x];
        for (unsigned j = info.x + 1; j < info.x + info.y; ++j) {
            const double4 p = sbody[j];
            lo.x = fmin(lo.x, p.x); lo.y = fmin(lo.y, p.y); lo.z = fmin(lo.z, p.z);
            hi.x = fmax(hi.x, p.x); hi.y = fmax(hi.y, p.y); hi.z = fmax(hi.z, p.z);
            lo.w = fmax(lo.w, bsort[j]);
        }
        hi.w = 0.0;
        box_lo[t] = lo;
        box_hi[t] = hi;
        int p = nparent[t];
        while (p >= 0) {
            __threadfence();
            const uint4 pinfo = winfo[p];
            const int nch = (int)((pinfo.w >> 8) & 0xffu);
            if ((int)atomicAdd(&cnt[p], 1u) != nch - 1) break;   // siblings still pending
            __threadfence();
            const int f = (int)pinfo.z;
            lo = ldcg_d4(box_lo + f);
            hi = ldcg_d4(box_hi + f);
            for (int u = f + 1; u < f + nch; ++u) {
                const double4 a = ldcg_d4(box_lo + u), b = ldcg_d4(box_hi + u);
                lo.x = fmin(lo.x, a.x); lo.y = fmin(lo.y, a.y); lo.z = fmin(lo.z, a.z); lo.w = fmax(lo.w, a.w);
                hi.x = fmax(hi.x, b.x); hi.y = fmax(hi.y, b.y); hi.z = fmax(hi.z, b.z);
            }
            box_lo[p] = lo;
            box_hi[p] = hi;
            p = nparent[p];
        }
    }
}

constexpr int kBpWarps = 4;
constexpr int kBpStack = 1024;   // node ids per warp (a local search holds a few dozen)
constexpr int kBpRoom = kBpStack - 7 * kMaxLevel - 1;   // wide pops keep the stack below this (see the pop rule)
constexpr int kBpLeafQ = 96;     // surviving leaves waiting for their body tests

__device__ __forceinline__ double gap(double alo, double ahi, double blo, double bhi)
{
    // distance between the intervals [alo, ahi] and [blo, bhi] along one axis, one rounding
    return fmax(0.0, fmax(__dsub_rn(blo, ahi), __dsub_rn(alo, bhi)));
}

__global__ void __launch_bounds__(kBpWarps * 32)
broadphase_kernel(DevState *st, const unsigned *__restrict__ gstart, const double4 *__restrict__ sbody,
                  const double *__restrict__ bsort, const double *__restrict__ gbox,
                  const uint4 *__restrict__ winfo, const double4 *__restrict__ box_lo,
                  const double4 *__restrict__ box_hi, const unsigned *__restrict__ perm, int2 *__restrict__ pairs,
                  unsigned long long cap)
{
    __shared__ unsigned stack_all[kBpWarps][kBpStack];
    __shared__ unsigned leafq_all[kBpWarps][kBpLeafQ];
    const unsigned lane = lane_id(), warp = threadIdx.x >> 5;
    const unsigned lt = (1u << lane) - 1u;
    unsigned *stack = stack_all[warp];
    unsigned *leafq = leafq_all[warp];
    const unsigned ng = st->n_groups;
    const double ninf = __longlong_as_double(0xfff0000000000000ll);

    for (unsigned g = blockIdx.x * kBpWarps + warp; g < ng; g += gridDim.x * kBpWarps) {
        const unsigned gb = gstart[g], ge = gstart[g + 1];
        const unsigned a = gb + lane;
        const bool mine = a < ge;
        const double4 p = sbody[mine ? a : gb];
        const double ba = mine ? bsort[a] : ninf;
        const unsigned oa = perm[mine ? a : gb];
        double bg = ba;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) bg = fmax(bg, __shfl_xor_sync(0xffffffffu, bg, o));
        const double glx = gbox[6 * g + 0], gly = gbox[6 * g + 1], glz = gbox[6 * g + 2];
        const double ghx = gbox[6 * g + 3], ghy = gbox[6 * g + 4], ghz = gbox[6 * g + 5];

        unsigned top = 1, nleaf = 0;
        if (lane == 0) stack[0] = 0u;
        __syncwarp();
        while (true) {
            // ---- body tests of the queued leaves, when the queue may not take another batch or at the end ----
            if (nleaf > (unsigned)kBpLeafQ - 32u || (top == 0 && nleaf > 0)) {
                for (unsigned q = 0; q < nleaf; ++q) {
                    const uint4 info = winfo[leafq[q]];
                    const unsigned kb = info.x > gb ? info.x : gb;   // bodies before the group are found from their side
                    for (unsigned k = kb; k < info.x + info.y; ++k) {
                        const double4 s = sbody[k];
                        const double dx = __dsub_rn(s.x, p.x), dy = __dsub_rn(s.y, p.y), dz = __dsub_rn(s.z, p.z);
                        const double d2 = __fma_rn(dz, dz, __fma_rn(dy, dy, __dmul_rn(dx, dx)));
                        const double sr = __dadd_rn(ba, bsort[k]);
                        const bool hit = mine && k > a && d2 <= __dmul_rn(sr, sr);
                        const unsigned m = __ballot_sync(0xffffffffu, hit);
                        if (m) {
                            unsigned long long base = 0;
                            if (lane == (unsigned)(__ffs(m) - 1))
                                base = atomicAdd(&st->pair_count, (unsigned long long)__popc(m));
                            base = __shfl_sync(0xffffffffu, base, __ffs(m) - 1);
                            const unsigned long long at = base + __popc(m & lt);
                            if (hit && at < cap) {
                                const unsigned ok = perm[k];
                                pairs[at] = make_int2((int)(oa < ok ? oa : ok), (int)(oa < ok ? ok : oa));
                            }
                        }
                    }
                }
                nleaf = 0;
                __syncwarp();
            }
            if (top == 0) break;
            // ---- pop up to 32 nodes, one per lane ----
            // A pop of k nodes pushes at most 8k children, so k <= (kBpRoom - top) / 7 keeps the stack below
            // kBpRoom; when that allows fewer than two, the walk goes node by node (depth first), which adds at
            // most 7 entries per level below the popped node: <= 7 * 21 = 147 more.  The stack cannot overflow.
            unsigned take = top < 32u ? top : 32u;
            {
                const unsigned room = (unsigned)kBpRoom > top ? ((unsigned)kBpRoom - top) / 7u : 0u;
                if (take > room) take = room > 1u ? room : 1u;
            }
            top -= take;
            const bool have = lane < take;
            const unsigned t = have ? stack[top + lane] : 0u;
            __syncwarp();
            bool near = false, internal = false;
            unsigned first = 0, kids = 0;
            if (have) {
                const uint4 info = winfo[t];
                const double4 lo = box_lo[t], hi = box_hi[t];
                const double gx = gap(glx, ghx, lo.x, hi.x), gy = gap(gly, ghy, lo.y, hi.y), gz = gap(glz, ghz, lo.z, hi.z);
                const double d2 = __fma_rn(gz, gz, __fma_rn(gy, gy, __dmul_rn(gx, gx)));
                const double sr = __dadd_rn(bg, lo.w);
                near = (info.x + info.y > gb) && d2 <= __dmul_rn(sr, sr);
                internal = (int)info.z >= 0;
                first = info.z;
                kids = (info.w >> 8) & 0xffu;
            }
            // surviving leaves -> queue
            {
                const unsigned m = __ballot_sync(0xffffffffu, near && !internal);
                if (near && !internal) leafq[nleaf + __popc(m & lt)] = t;
                nleaf += __popc(m);
            }
            // surviving internal nodes -> their children onto the stack
            {
                const unsigned c = (near && internal) ? kids : 0u;
                unsigned inc = c;
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) {
                    const unsigned u = __shfl_up_sync(0xffffffffu, inc, o);
                    if (lane >= (unsigned)o) inc += u;
                }
                const unsigned total = __shfl_sync(0xffffffffu, inc, 31);
                if (top + total > (unsigned)kBpStack) {      // excluded by the pop rule above; stay memory-safe
                    if (lane == 0) atomicOr(&st->status, (int)kStatBpStack);
                } else {
                    for (unsigned u = 0; u < c; ++u) stack[top + inc - c + u] = first + u;
                    top += total;
                }
            }
            __syncwarp();
        }
    }
}

// ------------------------------------------------------------------------------------------ NEXT-4
__device__ __forceinline__ int uf_find(int *parent, int x)
{
    // path halving; parent[] only ever decreases along a chain, so concurrent hooks keep it a forest
    while (true) {
        const int p = ((volatile int *)parent)[x];
        if (p == x) return x;
        const int gp = ((volatile int *)parent)[p];
        if (gp != p) ((volatile int *)parent)[x] = gp;
        x = p;
    }
}

__global__ void uf_init_kernel(int *parent, int *size, double *mass, long long n)
{
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        parent[i] = (int)i;
        if (size) size[i] = 0;
        if (mass) mass[i] = 0.0;
    }
}

__global__ void uf_union_kernel(int *parent, const int2 *__restrict__ pairs, long long n_pairs, long long n,
                                DevState *st)
{
    for (long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x; e < n_pairs;
         e += (long long)gridDim.x * blockDim.x) {
        const int2 pr = pairs[e];
        if (pr.x < 0 || pr.y < 0 || pr.x >= n || pr.y >= n) {
            atomicAdd(&st->agg_counts[2], 1ull);   // reported as BH_ERR_INVALID_ARG
            continue;
        }
        int a = pr.x, b = pr.y;
        while (true) {
            a = uf_find(parent, a);
            b = uf_find(parent, b);
            if (a == b) break;
            if (a > b) { const int t = a; a = b; b = t; }
            if (atomicCAS(&parent[b], b, a) == b) break;    // hook the larger root under the smaller
        }
    }
}

__global__ void uf_flatten_kernel(int *parent, int *size, double *mass, const double *__restrict__ mass_in,
                                  long long n)
{
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        int r = (int)i;
        while (true) {   // no hooks are in flight any more: plain chase to the root
            const int p = parent[r];
            if (p == r) break;
            r = p;
        }
        // writing the root to parent[i] while other threads still chase through i is harmless: every
        // value ever stored is an ancestor of i
        ((volatile int *)parent)[i] = r;
        if (size) atomicAdd(&size[r], 1);
        if (mass && mass_in) atomicAdd(&mass[r], mass_in[i]);
    }
}

__global__ void uf_count_kernel(const int *__restrict__ label, const int *__restrict__ size, long long n,
                                unsigned long long *counts)
{
    unsigned long long comps = 0, aggs = 0;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        if (label[i] == (int)i) {
            ++comps;
            if (size[i] > 1) ++aggs;
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        comps += __shfl_xor_sync(0xffffffffu, comps, o);
        aggs += __shfl_xor_sync(0xffffffffu, aggs, o);
    }
    if (lane_id() == 0 && comps) {
        atomicAdd(&counts[0], comps);
        if (aggs) atomicAdd(&counts[1], aggs);
    }
}

// ------------------------------------------------------------------------------------------ launchers
int launch_broadphase(const Workspace &w, int64_t n, const double *radius, const double *vel, double dt,
                      int32_t *pairs, int64_t cap, cudaStream_t s)
{
    cudaMemsetAsync(w.bp_cnt, 0, (size_t)node_capacity(n, w.leaf_cap) * sizeof(unsigned), s);
    cudaMemsetAsync(&w.st->pair_count, 0, sizeof(unsigned long long), s);
    bound_radius_kernel<<<(int)((n + 255) / 256), 256, 0, s>>>(radius, vel, w.idx[0], n, dt, w.bsort);
    const int64_t want = (node_capacity(n, w.leaf_cap) + 255) / 256;
    node_box_kernel<<<(int)(want < w.sms * 16 ? want : w.sms * 16), 256, 0, s>>>(w.st, w.sbody, w.bsort, w.winfo, w.nparent,
                                                                             w.bp_cnt, w.box_lo, w.box_hi, w.node_cap);
    broadphase_kernel<<<w.sms * 16, kBpWarps * 32, 0, s>>>(w.st, w.gstart, w.sbody, w.bsort, w.gbox, w.winfo, w.box_lo,
                                                        w.box_hi, w.idx[0], reinterpret_cast<int2 *>(pairs),
                                                        (unsigned long long)cap);
    return 3;
}

int launch_aggregates(const Workspace &w, int64_t n, const int32_t *pairs, int64_t n_pairs, const double *mass_in,
                      int32_t *label, int32_t *size, double *mass, cudaStream_t s)
{
    cudaMemsetAsync(w.st->agg_counts, 0, 3 * sizeof(unsigned long long), s);
    if (!size) size = w.agg_size;
    const int nb = (int)((n + 255) / 256 < w.sms * 8 ? (n + 255) / 256 : w.sms * 8);
    uf_init_kernel<<<nb, 256, 0, s>>>(label, size, mass, n);
    int launches = 3;
    if (n_pairs > 0) {
        const int pb = (int)((n_pairs + 255) / 256 < w.sms * 16 ? (n_pairs + 255) / 256 : w.sms * 16);
        uf_union_kernel<<<pb, 256, 0, s>>>(label, reinterpret_cast<const int2 *>(pairs), n_pairs, n, w.st);
        ++launches;
    }
    uf_flatten_kernel<<<nb, 256, 0, s>>>(label, size, mass, mass_in, n);
    uf_count_kernel<<<nb, 256, 0, s>>>(label, size, n, w.st->agg_counts);
    return launches;
}

}  // namespace bh
