// bh_diag.cu — rows "next" of SURVEY.md §8(f), NEXT-1 / NEXT-2: conserved quantities (PAPER.md:176, 186:
// energy, linear and angular momentum of the purely gravitational system), the maximum relative position
// error of Eq. (7), and the update kernel of the paper's preferred semi-implicit Euler
// stepper and of its two-rate scheme.
//
// Conserved quantities are sums with heavy cancellation (the total momentum of an equilibrium cloud is
// ~0), so every thread accumulates in double-double (error-free products by fma, two-sum additions) and
// the partial sums are combined in a fixed order: per warp by shuffles, per block through shared
// memory, and by the last block to finish (ticket) over the per-block results in block order.  The
// result does not depend on scheduling and is good to ~1e-30 relative to the sum of |terms|, then
// rounded once to fp64.
#include <cstdio>
#include <mutex>

#include "bh_common.cuh"

namespace bh {

struct dd {
    double hi, lo;
};

__device__ __forceinline__ dd two_sum(double a, double b)
{
    const double s = __dadd_rn(a, b);
    const double bb = __dsub_rn(s, a);
    const double e = __dadd_rn(__dsub_rn(a, __dsub_rn(s, bb)), __dsub_rn(b, bb));
    return {s, e};
}
__device__ __forceinline__ dd two_prod(double a, double b)
{
    const double p = __dmul_rn(a, b);
    return {p, __fma_rn(a, b, -p)};
}
__device__ __forceinline__ dd dd_add(dd a, dd b)
{
    dd s = two_sum(a.hi, b.hi);
    const double e = __dadd_rn(s.lo, __dadd_rn(a.lo, b.lo));
    const double h = __dadd_rn(s.hi, e);
    return {h, __dsub_rn(e, __dsub_rn(h, s.hi))};
}
__device__ __forceinline__ dd dd_mul_d(dd a, double b)   // (a.hi + a.lo) * b
{
    dd p = two_prod(a.hi, b);
    const double e = __fma_rn(a.lo, b, p.lo);
    const double h = __dadd_rn(p.hi, e);
    return {h, __dsub_rn(e, __dsub_rn(h, p.hi))};
}
__device__ __forceinline__ dd dd_sub(dd a, dd b) { return dd_add(a, {-b.hi, -b.lo}); }

constexpr int kDiagThreads = 256;
constexpr int kDiagQ = 8;   // ekin, epot, Px, Py, Pz, Lx, Ly, Lz

// out: [0..7] the eight sums rounded to fp64.  part: [blocks][8][2] per-block double-double partials.
__global__ void __launch_bounds__(kDiagThreads)
diag_kernel(const double *__restrict__ pos, const double *__restrict__ vel, const double *__restrict__ mass,
            const double *__restrict__ phi, long long n, double *__restrict__ part, unsigned *ticket,
            double *__restrict__ out)
{
    dd acc[kDiagQ];
#pragma unroll
    for (int q = 0; q < kDiagQ; ++q) acc[q] = {0.0, 0.0};
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        const double m = mass[i];
        const double x = pos[3 * i], y = pos[3 * i + 1], z = pos[3 * i + 2];
        const double vx = vel[3 * i], vy = vel[3 * i + 1], vz = vel[3 * i + 2];
        // kinetic energy 1/2 m |v|^2: |v|^2 as a double-double sum of exact squares
        dd v2 = dd_add(dd_add(two_prod(vx, vx), two_prod(vy, vy)), two_prod(vz, vz));
        acc[0] = dd_add(acc[0], dd_mul_d(v2, 0.5 * m));
        if (phi) acc[1] = dd_add(acc[1], two_prod(0.5 * m, phi[i]));
        acc[2] = dd_add(acc[2], two_prod(m, vx));
        acc[3] = dd_add(acc[3], two_prod(m, vy));
        acc[4] = dd_add(acc[4], two_prod(m, vz));
        acc[5] = dd_add(acc[5], dd_mul_d(dd_sub(two_prod(y, vz), two_prod(z, vy)), m));
        acc[6] = dd_add(acc[6], dd_mul_d(dd_sub(two_prod(z, vx), two_prod(x, vz)), m));
        acc[7] = dd_add(acc[7], dd_mul_d(dd_sub(two_prod(x, vy), two_prod(y, vx)), m));
    }
    __shared__ double sh[kDiagThreads / 32][kDiagQ][2];
    __shared__ bool last;
    const unsigned lane = lane_id(), warp = threadIdx.x >> 5;
#pragma unroll
    for (int q = 0; q < kDiagQ; ++q) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            dd other = {__shfl_down_sync(0xffffffffu, acc[q].hi, o), __shfl_down_sync(0xffffffffu, acc[q].lo, o)};
            acc[q] = dd_add(acc[q], other);
        }
        if (lane == 0) {
            sh[warp][q][0] = acc[q].hi;
            sh[warp][q][1] = acc[q].lo;
        }
    }
    __syncthreads();
    if (threadIdx.x < kDiagQ) {
        const int q = threadIdx.x;
        dd s = {sh[0][q][0], sh[0][q][1]};
        for (int w = 1; w < kDiagThreads / 32; ++w) s = dd_add(s, {sh[w][q][0], sh[w][q][1]});
        part[((size_t)blockIdx.x * kDiagQ + q) * 2 + 0] = s.hi;
        part[((size_t)blockIdx.x * kDiagQ + q) * 2 + 1] = s.lo;
        __threadfence();
    }
    __syncthreads();
    if (threadIdx.x == 0) last = atomicAdd(ticket, 1u) == gridDim.x - 1;
    __syncthreads();
    if (last) {
        // the last block adds the per-block partials in a fixed order: lane j of warp q takes blocks j, j + 32, ...
        // in increasing order, then the 32 lane sums are added in lane order (warp q = quantity q)
        __threadfence();
        const int q = threadIdx.x >> 5;
        const volatile double *vp = part;
        dd s = {0.0, 0.0};
        for (unsigned b = lane; b < gridDim.x; b += 32)
            s = dd_add(s, {vp[((size_t)b * kDiagQ + q) * 2 + 0], vp[((size_t)b * kDiagQ + q) * 2 + 1]});
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            dd other = {__shfl_down_sync(0xffffffffu, s.hi, o), __shfl_down_sync(0xffffffffu, s.lo, o)};
            s = dd_add(s, other);
        }
        if (lane == 0) out[q] = s.hi;
        if (threadIdx.x == 0) *ticket = 0u;
    }
}

// Eq. (7): e_i = 100 sqrt(|r - r_ref|^2 / |r_ref|^2), canonical arithmetic (every operation IEEE-rounded
// once, |.|^2 = fma(z, z, fma(y, y, x*x))); bodies whose reference position is the origin are skipped
// (R25).  Non-negative doubles order like their bit patterns, so the maximum is an integer atomicMax.
__global__ void __launch_bounds__(256)
poserr_kernel(const double *__restrict__ pos, const double *__restrict__ ref, long long n, unsigned long long *out_bits)
{
    double worst = 0.0;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        const double rx = ref[3 * i], ry = ref[3 * i + 1], rz = ref[3 * i + 2];
        const double dx = __dsub_rn(pos[3 * i], rx), dy = __dsub_rn(pos[3 * i + 1], ry), dz = __dsub_rn(pos[3 * i + 2], rz);
        const double nd = __fma_rn(dz, dz, __fma_rn(dy, dy, __dmul_rn(dx, dx)));
        const double nr = __fma_rn(rz, rz, __fma_rn(ry, ry, __dmul_rn(rx, rx)));
        if (nr == 0.0) continue;
        const double e = __dmul_rn(100.0, __dsqrt_rn(__ddiv_rn(nd, nr)));
        if (e > worst) worst = e;   // a NaN (non-finite input) never wins, as in a plain comparison
    }
    unsigned long long b = (unsigned long long)__double_as_longlong(worst);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        const unsigned long long t = __shfl_xor_sync(0xffffffffu, b, o);
        b = t > b ? t : b;
    }
    if (lane_id() == 0 && b) atomicMax(out_bits, b);
}

// n_sub semi-implicit Euler sub-steps with one, constant acceleration (n_sub = 1 is
// the plain stepper of PAPER.md:148): v = fma(a, dt, v); x = fma(v, dt, x), repeated in registers —
// bit-identical to n_sub separate passes, one trip through HBM.
__global__ void euler_sub_kernel(double *__restrict__ pos, double *__restrict__ vel, const double *__restrict__ acc,
                                 long long n3, double dt, int n_sub)
{
    for (long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x; k < n3;
         k += (long long)gridDim.x * blockDim.x) {
        const double a = acc[k];
        double v = vel[k], x = pos[k];
        for (int q = 0; q < n_sub; ++q) {
            v = __fma_rn(a, dt, v);
            x = __fma_rn(v, dt, x);
        }
        vel[k] = v;
        pos[k] = x;
    }
}

void launch_diagnostics(const Workspace &w, const double *pos, const double *vel, const double *mass,
                        const double *phi, int64_t n, cudaStream_t s)
{
    int blocks = (int)((n + kDiagThreads - 1) / kDiagThreads);
    if (blocks > kDiagBlocks) blocks = kDiagBlocks;
    diag_kernel<<<blocks, kDiagThreads, 0, s>>>(pos, vel, mass, phi, n, w.diag_part, w.diag_ticket, w.diag_out);
}

void launch_position_error(const Workspace &w, const double *pos, const double *ref, int64_t n, cudaStream_t s)
{
    cudaMemsetAsync(w.diag_out + kDiagQ, 0, sizeof(double), s);
    int blocks = (int)((n + 255) / 256);
    if (blocks > w.sms * 8) blocks = w.sms * 8;
    poserr_kernel<<<blocks, 256, 0, s>>>(pos, ref, n, reinterpret_cast<unsigned long long *>(w.diag_out + kDiagQ));
}

void launch_euler_sub(double *pos, double *vel, const double *acc, int64_t n, double dt, int n_sub, cudaStream_t s)
{
    const long long n3 = 3ll * n;
    int blocks = (int)((n3 + 1023) / 1024);
    if (blocks > sm_count() * 8) blocks = sm_count() * 8;
    euler_sub_kernel<<<blocks, 256, 0, s>>>(pos, vel, acc, n3, dt, n_sub);
}

// ---- bh_diagnostics_static: the conserved quantities without a context, a workspace or any allocation ----
//
// diag_kernel needs scratch memory: one row of eight double-double partial sums per block, and the ticket
// that elects the block which adds the rows up.  bh_diagnostics takes both from the workspace the caller
// allocated for bh_create.  The scratch below lives in the library image instead, so a caller that owns no
// device allocator at all can still follow the energy and momenta of bodies somebody else keeps on the GPU.
// Row layout as in diag_kernel: [block][quantity][hi, lo]; the ticket sits in a 256-byte row of its own
// after the last partial row.
constexpr size_t kStaticDiagPartDoubles = (size_t)kDiagBlocks * kDiagQ * 2;          // 592 x 8 x 2 doubles = 75 776 bytes
constexpr size_t kStaticDiagDoubles = kStaticDiagPartDoubles + 256 / sizeof(double);   // + the ticket's row
static_assert(kStaticDiagDoubles * sizeof(double) == BH_DIAG_STATIC_SCRATCH_BYTES, "bh.h states the size of the static scratch");

static __device__ __align__(256) double g_static_diag_scratch[kStaticDiagDoubles];

constexpr int kStaticMaxDevices = 64;
static double *g_static_diag_ptr[kStaticMaxDevices];   // device address of the array, per device ordinal; null = not asked yet
static std::mutex g_static_diag_mutex;

// Address of g_static_diag_scratch on the CURRENT device.  In host code the array's name is only the handle
// the runtime registered for it, not somewhere a kernel can read or write: the real address differs from GPU
// to GPU and has to be asked for with that GPU current, once.
static cudaError_t static_diag_scratch(double **out)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= kStaticMaxDevices) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> hold(g_static_diag_mutex);
    if (!g_static_diag_ptr[dev]) {
        void *p = nullptr;
        e = cudaGetSymbolAddress(&p, g_static_diag_scratch);
        if (e != cudaSuccess) return e;
        g_static_diag_ptr[dev] = static_cast<double *>(p);
    }
    *out = g_static_diag_ptr[dev];
    return cudaSuccess;
}

}  // namespace bh

extern "C" bh_status bh_diagnostics_static(const double *pos_dev, const double *vel_dev, const double *mass_dev,
                                           const double *phi_dev, int64_t n, double *out_dev, void *cuda_stream)
{
    using namespace bh;
    char msg[256];
    if (!pos_dev || !vel_dev || !mass_dev || !out_dev) {
        set_global_error("bh_diagnostics_static: null pointer");
        return BH_ERR_INVALID_ARG;
    }
    if (n < 1) {
        set_global_error("bh_diagnostics_static: n < 1");
        return BH_ERR_INVALID_ARG;
    }
    if (n > BH_DIAG_STATIC_MAX_N) {
        snprintf(msg, sizeof msg, "bh_diagnostics_static: n = %lld is above BH_DIAG_STATIC_MAX_N = %lld, the most bodies "
                 "the fixed scratch array is specified for (use bh_diagnostics with a workspace)",
                 (long long)n, (long long)BH_DIAG_STATIC_MAX_N);
        set_global_error(msg);
        return BH_ERR_CAPACITY;
    }
    double *scratch = nullptr;
    cudaError_t e = static_diag_scratch(&scratch);
    if (e != cudaSuccess) {
        snprintf(msg, sizeof msg, "bh_diagnostics_static: address of the static scratch: %s", cudaGetErrorString(e));
        set_global_error(msg);
        return BH_ERR_CUDA;
    }
    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
    unsigned *ticket = reinterpret_cast<unsigned *>(scratch + kStaticDiagPartDoubles);
    // The ticket must read 0 when the first block arrives.  A completed call leaves it at 0, but the array is
    // shared by everybody in the process, so a call that was cut short (a fault, a reset stream) may not have:
    // clear it every time.  The partial rows need no clearing: a block writes its row before it takes a ticket,
    // and only rows of this launch's blocks are read.
    e = cudaMemsetAsync(ticket, 0, sizeof(unsigned), s);
    if (e == cudaSuccess) {
        // same grid as launch_diagnostics: the rows, and with them the order of the additions, are those of
        // bh_diagnostics, so the two calls give the same bits
        int blocks = (int)((n + kDiagThreads - 1) / kDiagThreads);
        if (blocks > kDiagBlocks) blocks = kDiagBlocks;
        diag_kernel<<<blocks, kDiagThreads, 0, s>>>(pos_dev, vel_dev, mass_dev, phi_dev, n, scratch, ticket, out_dev);
        e = cudaGetLastError();
    }
    if (e != cudaSuccess) {
        snprintf(msg, sizeof msg, "bh_diagnostics_static launch: %s", cudaGetErrorString(e));
        set_global_error(msg);
        return BH_ERR_CUDA;
    }
    return BH_OK;
}
