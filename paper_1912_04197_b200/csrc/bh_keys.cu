// bh_keys.cu — step a1 (canonical bounding cube) and step a2 (63-bit Morton keys over
// that cube, plus the digit histograms of all eight radix passes).  HBM-streaming kernels.
#include "bh_keys.cuh"

namespace bh {

constexpr int kCubeThreads = 192;   // multiple of 3: a thread always sees the same axis

// The block's share of the extremes (thread t only ever met axis t % 3) -> part[blk][8]; the last block to finish reduces
// the partials and derives the cube (finish_cube).  Shared by cube_kernel and kick_drift_cube_kernel.
__device__ __forceinline__ void cube_block_finish(double mn, double mx, int bad, DevState *st, double *part, double *smn,
                                                  double *smx, int *sbad, bool *is_last_p)
{
    const int tid = threadIdx.x;
    smn[tid] = mn;
    smx[tid] = mx;
    sbad[tid] = bad;
    __syncthreads();
    // tree over strides that are multiples of 3, so that a thread only ever meets its own axis
#pragma unroll
    for (int h = kCubeThreads / 2; h >= 3; h >>= 1) {
        if (tid < h) {
            smn[tid] = fmin(smn[tid], smn[tid + h]);
            smx[tid] = fmax(smx[tid], smx[tid + h]);
            sbad[tid] |= sbad[tid + h];
        }
        __syncthreads();
    }
    if (tid < 3) {
        part[blockIdx.x * 8 + tid] = smn[tid];
        part[blockIdx.x * 8 + 3 + tid] = smx[tid];
    }
    if (tid == 0) part[blockIdx.x * 8 + 6] = (sbad[0] | sbad[1] | sbad[2]) ? 1.0 : 0.0;
    __threadfence();
    __syncthreads();
    if (tid == 0) *is_last_p = (atomicAdd(&st->ticket_bbox, 1u) == gridDim.x - 1);
    __syncthreads();
    if (!*is_last_p) return;
    __threadfence();
    // final reduction over blocks: thread t takes axis t%3 of blocks t/3, t/3+64, ...
    const int axis = tid % 3;
    mn = __longlong_as_double(0x7ff0000000000000ll);
    mx = -mn;
    bad = 0;
    for (int b = tid / 3; b < (int)gridDim.x; b += kCubeThreads / 3) {
        mn = fmin(mn, __ldcg(part + b * 8 + axis));
        mx = fmax(mx, __ldcg(part + b * 8 + 3 + axis));
        bad |= (__ldcg(part + b * 8 + 6) != 0.0);
    }
    smn[tid] = mn;
    smx[tid] = mx;
    sbad[tid] = bad;
    __syncthreads();
#pragma unroll
    for (int h = kCubeThreads / 2; h >= 3; h >>= 1) {
        if (tid < h) {
            smn[tid] = fmin(smn[tid], smn[tid + h]);
            smx[tid] = fmax(smx[tid], smx[tid + h]);
            sbad[tid] |= sbad[tid + h];
        }
        __syncthreads();
    }
    if (tid == 0) {
        double lo[3], hi[3];
        for (int a = 0; a < 3; ++a) {
            lo[a] = smn[a];
            hi[a] = smx[a];
        }
        finish_cube(lo, hi, sbad[0] | sbad[1] | sbad[2], st);
    }
}

// What a streaming build clears before its first kernel needs it (histograms and tickets + the look-back rows of this n;
// child masks / arrival counters of the nodes n bodies can make): done by the first kernel of the build, grid-wide,
// instead of two memsets in front of it.
struct BuildClear {
    uint4 *a;
    long long a16;      // 16-byte words
    uint4 *b;
    long long b16;
};
__device__ __forceinline__ void clear_for_build(const BuildClear &z)
{
    const long long g = (long long)blockIdx.x * blockDim.x + threadIdx.x, step = (long long)gridDim.x * blockDim.x;
    const uint4 zero = make_uint4(0u, 0u, 0u, 0u);
    for (long long k = g; k < z.a16; k += step) z.a[k] = zero;
    for (long long k = g; k < z.b16; k += step) z.b[k] = zero;
}
static BuildClear build_clear(const Workspace &w, int64_t n)
{
    const int64_t tile_keys = (int64_t)kSortThreads * sort_tile_items(n);
    const int64_t tiles = (n + tile_keys - 1) / tile_keys;
    const size_t abytes = (size_t)((char *)w.lookback - (char *)w.zero_begin) + (size_t)kSortPasses * tiles * kRadix * sizeof(unsigned);
    const size_t bbytes = (size_t)node_capacity(n, w.leaf_cap) * sizeof(unsigned);
    BuildClear z;
    z.a = reinterpret_cast<uint4 *>(w.zero_begin);
    z.a16 = (long long)((abytes + 15) / 16);
    z.b = reinterpret_cast<uint4 *>(w.node_meta);
    z.b16 = (long long)((bbytes + 15) / 16);
    return z;
}

// One pass over the flat [3n] coordinate array; per-block partial (min, max, bad) to part[blk][8];
// the last block to finish reduces the partials and derives the cube (R11): corner = per-axis
// minimum, side = smallest power of two strictly above the largest extent (1 if the extent is 0).
__global__ void __launch_bounds__(kCubeThreads) cube_kernel(const double *__restrict__ pos, long long n3,
                                                            DevState *st, double *part, BuildClear zc)
{
    clear_for_build(zc);
    __shared__ double smn[kCubeThreads], smx[kCubeThreads];
    __shared__ int sbad[kCubeThreads];
    __shared__ bool is_last;
    const int tid = threadIdx.x;
    const long long stride = (long long)gridDim.x * kCubeThreads;
    double mn = __longlong_as_double(0x7ff0000000000000ll), mx = -mn;
    int bad = 0;
    // four independent loads in flight per thread (the stride is a multiple of 3: same axis)
    long long k = (long long)blockIdx.x * kCubeThreads + tid;
    for (; k + 3 * stride < n3; k += 4 * stride) {
        const double x0 = __ldg(pos + k), x1 = __ldg(pos + k + stride), x2 = __ldg(pos + k + 2 * stride),
                     x3 = __ldg(pos + k + 3 * stride);
        bad |= nonfinite(x0) | nonfinite(x1) | nonfinite(x2) | nonfinite(x3);
        mn = fmin(fmin(mn, x0), fmin(x1, fmin(x2, x3)));
        mx = fmax(fmax(mx, x0), fmax(x1, fmax(x2, x3)));
    }
    for (; k < n3; k += stride) {
        double x = __ldg(pos + k);
        bad |= nonfinite(x);
        mn = fmin(mn, x);
        mx = fmax(mx, x);
    }
    cube_block_finish(mn, mx, bad, st, part, smn, smx, sbad, &is_last);
}

// Leapfrog kick + drift (R18) and the bounding cube of the NEW positions in one pass: v <- fma(a, dt/2, v); x <- fma(v, dt, x)
// — the arithmetic of kick_drift_kernel — and the extremes of x as cube_kernel takes them, so that the build that follows
// a step's drift needs no pass of its own over the positions.
__global__ void __launch_bounds__(kCubeThreads) kick_drift_cube_kernel(double *__restrict__ pos, double *__restrict__ vel,
                                                                       const double *__restrict__ acc, long long n3,
                                                                       double h, double dt, DevState *st, double *part,
                                                                       BuildClear zc)
{
    clear_for_build(zc);
    __shared__ double smn[kCubeThreads], smx[kCubeThreads];
    __shared__ int sbad[kCubeThreads];
    __shared__ bool is_last;
    const long long stride = (long long)gridDim.x * kCubeThreads;     // a multiple of 3: a thread keeps its axis
    double mn = __longlong_as_double(0x7ff0000000000000ll), mx = -mn;
    int bad = 0;
    // four elements per trip, their twelve loads issued together
    long long k = (long long)blockIdx.x * kCubeThreads + threadIdx.x;
    for (; k + 3 * stride < n3; k += 4 * stride) {
        double a[4], v[4], x[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            a[u] = acc[k + u * stride];
            v[u] = vel[k + u * stride];
            x[u] = pos[k + u * stride];
        }
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            v[u] = __fma_rn(a[u], h, v[u]);
            x[u] = __fma_rn(v[u], dt, x[u]);
            vel[k + u * stride] = v[u];
            pos[k + u * stride] = x[u];
            bad |= nonfinite(x[u]);
            mn = fmin(mn, x[u]);
            mx = fmax(mx, x[u]);
        }
    }
    for (; k < n3; k += stride) {
        const double v = __fma_rn(acc[k], h, vel[k]);
        vel[k] = v;
        const double x = __fma_rn(v, dt, pos[k]);
        pos[k] = x;
        bad |= nonfinite(x);
        mn = fmin(mn, x);
        mx = fmax(mx, x);
    }
    cube_block_finish(mn, mx, bad, st, part, smn, smx, sbad, &is_last);
}

// keys + the 8 x 256 digit histograms (shared-memory atomics, flushed once per block)
__global__ void __launch_bounds__(256) keys_kernel(const double *__restrict__ pos, long long n,
                                                   const DevState *__restrict__ st,
                                                   unsigned long long *__restrict__ key,
                                                   unsigned *__restrict__ hist)
{
    __shared__ unsigned sh[kSortPasses * kRadix];
    for (int k = threadIdx.x; k < kSortPasses * kRadix; k += blockDim.x) sh[k] = 0u;
    __syncthreads();
    const double lx = st->lo[0], ly = st->lo[1], lz = st->lo[2], sc = st->scale;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n;
         i += (long long)gridDim.x * blockDim.x) {
        const unsigned long long k = morton_key(__ldg(pos + 3 * i + 0), __ldg(pos + 3 * i + 1), __ldg(pos + 3 * i + 2), lx, ly, lz, sc);
        key[i] = k;
#pragma unroll
        for (int p = 0; p < kSortPasses; ++p)
            atomicAdd(&sh[p * kRadix + (unsigned)((k >> (p * kRadixBits)) & (kRadix - 1))], 1u);
    }
    __syncthreads();
    for (int k = threadIdx.x; k < kSortPasses * kRadix; k += blockDim.x)
        if (sh[k]) atomicAdd(&hist[k], sh[k]);
}

void launch_cube(const Workspace &w, const double *pos, int64_t n, cudaStream_t s)
{
    long long n3 = 3 * (long long)n;
    int blocks = (int)((n3 + kCubeThreads * 4 - 1) / (kCubeThreads * 4));   // four loads per thread, all in flight
    if (blocks > w.sms * 4) blocks = w.sms * 4;   // bbox_part holds kMaxBboxBlocks rows
    if (blocks > kMaxBboxBlocks) blocks = kMaxBboxBlocks;
    if (blocks < 1) blocks = 1;
    cube_kernel<<<blocks, kCubeThreads, 0, s>>>(pos, n3, w.st, w.bbox_part, build_clear(w, n));
}

void launch_kick_drift_cube(const Workspace &w, double *pos, double *vel, const double *acc, int64_t n, double dt,
                            cudaStream_t s)
{
    long long n3 = 3 * (long long)n;
    int blocks = (int)((n3 + kCubeThreads * 4 - 1) / (kCubeThreads * 4));
    if (blocks > w.sms * 4) blocks = w.sms * 4;   // bbox_part holds kMaxBboxBlocks rows
    if (blocks > kMaxBboxBlocks) blocks = kMaxBboxBlocks;
    if (blocks < 1) blocks = 1;
    kick_drift_cube_kernel<<<blocks, kCubeThreads, 0, s>>>(pos, vel, acc, n3, dt * 0.5, dt, w.st, w.bbox_part, build_clear(w, n));
}

void launch_keys(const Workspace &w, const double *pos, int64_t n, cudaStream_t s)
{
    int blocks = (int)((n + 256 * 4 - 1) / (256 * 4));
    if (blocks > w.sms * 8) blocks = w.sms * 8;
    if (blocks < 1) blocks = 1;
    keys_kernel<<<blocks, 256, 0, s>>>(pos, n, w.st, w.key[0], w.hist);
}

}  // namespace bh
