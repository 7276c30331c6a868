// bh_microbench.cu — measurement-only kernels behind bench.py's roofline statement (NOT part of libbh):
//   bhmb_fp64_peak     register-resident DFMA chains on every SM: the measured fp64 FMA rate, the roofline
//                      denominator of the walk (a7) and direct (a8) kernels (MEASURED_PEAKS.json has no fp64 entry);
//   bhmb_issue_model   the walk's own evaluation loop (bh_eval.cuh) alone on a sub-partition and beside
//                      integer-issuing warps: what a warp-specialised walk can reach.
//   bhmb_fp64_mma      the fp64 tensor-core MMA (mma.sync m8n8k4 f64 = DMMA.8) alone and interleaved with DFMA
//                      chains: on sm_100 it runs at the vector fp64 rate AND on the same datapath (times add),
//                      so recasting r^2 or the accumulation as a contraction cannot relieve the fp64 pipe.
// Built into libbh_microbench.so by paper_1912_04197_b200/build.py; loaded by bench.py only.
#include "../bh_eval.cuh"

namespace bh {

// ------------------------------------------------------------------------------------------ fp64 peak
__global__ void __launch_bounds__(256) fp64_peak_kernel(double *sink, int iters, double seed)
{
    double a0 = seed + threadIdx.x, a1 = a0 + 1, a2 = a0 + 2, a3 = a0 + 3, a4 = a0 + 4, a5 = a0 + 5, a6 = a0 + 6,
           a7 = a0 + 7;
    const double m = 0.999999, c = 1e-9;
    // sixteen trips per branch: the loop's own integer instructions take issue slots from the DFMAs of the same
    // sub-partition (34.8 TFLOP/s without the unroll against 36.0 with it, same chip, same minute)
#pragma unroll 16
    for (int i = 0; i < iters; ++i) {
        a0 = fma(a0, m, c); a1 = fma(a1, m, c); a2 = fma(a2, m, c); a3 = fma(a3, m, c);
        a4 = fma(a4, m, c); a5 = fma(a5, m, c); a6 = fma(a6, m, c); a7 = fma(a7, m, c);
    }
    double s = a0 + a1 + a2 + a3 + a4 + a5 + a6 + a7;
    if (s == 123456.789) sink[0] = s;
}

// ------------------------------------------------------------------------------------------ issue model
// What the walk's evaluation loop reaches when nothing else runs on its sub-partition, and what it loses to
// co-resident warps that issue integer / shared-memory instructions (as the walk's producer warps do).  Same
// block shape as walk_kernel: 16 warps, warps 4-7 and 12-15 evaluate (two per sub-partition, four bodies per
// lane, sources from a 512-entry shared-memory ring); the other eight warps exit (HOG 0), run a dependent
// IMAD / LDS chain at low duty (HOG 1) or independent IMADs at full rate (HOG 2) until the evaluators are done.
template <int HOG>
__global__ void __launch_bounds__(512, 1) issue_model_kernel(double *sink, int iters, double eps2, int seed)
{
    __shared__ double4 ring[512];
    __shared__ int tab[1024];
    __shared__ int done;
    for (int i = threadIdx.x; i < 512; i += blockDim.x) ring[i] = make_double4(1.0 + i * 0.01, 2.0 - i * 0.02, 0.5 + i * 0.003, 1e-3);
    for (int i = threadIdx.x; i < 1024; i += blockDim.x) tab[i] = (i * 7 + seed) & 1023;
    if (threadIdx.x == 0) done = 0;
    __syncthreads();
    const unsigned warp = threadIdx.x >> 5, lane = threadIdx.x & 31u, quarter = lane >> 3;
    if (((warp >> 2) & 1u) == 1u) {
        Bodies<4> B;
        for (int s = 0; s < 4; ++s) {
            B.x[s] = 0.1 * lane + s; B.y[s] = 0.2 * s; B.z[s] = 0.05 * lane;
            B.ax[s] = B.ay[s] = B.az[s] = B.ph[s] = 0.0;
        }
        for (int it = 0; it < iters; ++it) eval_blocks<false, 4, 0>(ring, 0u, 512u, quarter, eps2, B);
        double s = 0.0;
        for (int q = 0; q < 4; ++q) s += B.ax[q] + B.ay[q] + B.az[q];
        if (s == 123.456) sink[0] = s;
        __syncwarp();
        if (lane == 0) atomicAdd(&done, 1);
    } else if (HOG != 0) {
        int a = seed + (int)lane, b = seed * 3 + (int)lane, c = (int)lane;
        while (*((volatile int *)&done) < 8) {
            if (HOG == 1) {
                for (int r = 0; r < 16; ++r) { a = tab[(a * 5 + b) & 1023]; b = b * 3 + a; c ^= a + b; }
            } else {
                for (int r = 0; r < 16; ++r) { a = a * 5 + seed; b = b * 3 + seed; c = c * 7 + seed; }
            }
        }
        if (a + b + c == 12345) sink[1] = a;
    }
}


// MODE 0: eight DFMA chains per thread; 1: eight independent m8n8k4 f64 MMAs per warp; 2: both interleaved
template <int MODE>
__global__ void __launch_bounds__(256) fp64_mma_kernel(double *sink, int iters, double seed)
{
    double f[8], c[8][2];
    const double m = 0.999999, q = 1e-9;
    for (int i = 0; i < 8; ++i) { f[i] = seed + threadIdx.x + i; c[i][0] = seed * i; c[i][1] = seed + i; }
    const double a = seed * 1e-3 + threadIdx.x * 1e-6, b = 1e-3;
    for (int it = 0; it < iters; ++it) {
        if (MODE != 1) {
#pragma unroll
            for (int i = 0; i < 8; ++i) f[i] = fma(f[i], m, q);
        }
        if (MODE != 0) {
#pragma unroll
            for (int i = 0; i < 8; ++i)
                asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                             : "+d"(c[i][0]), "+d"(c[i][1]) : "d"(a), "d"(b));
        }
    }
    double s = 0;
    for (int i = 0; i < 8; ++i) s += f[i] + c[i][0] + c[i][1];
    if (s == 123456.789) sink[0] = s;
}

template <int MODE>
static float run_fp64_mma_one(double *sink, int blocks, int iters, cudaStream_t s)
{
    cudaEvent_t a, b;
    cudaEventCreate(&a);
    cudaEventCreate(&b);
    fp64_mma_kernel<MODE><<<blocks, 256, 0, s>>>(sink, 64, 1.0);
    cudaEventRecord(a, s);
    fp64_mma_kernel<MODE><<<blocks, 256, 0, s>>>(sink, iters, 1.0);
    cudaEventRecord(b, s);
    cudaEventSynchronize(b);
    float ms = 0.f;
    cudaEventElapsedTime(&ms, a, b);
    cudaEventDestroy(a);
    cudaEventDestroy(b);
    return ms;
}

static int device_sms()
{
    int dev = 0, v = kDefaultSMs;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&v, cudaDevAttrMultiProcessorCount, dev);
    return v;
}

template <int HOG>
static double run_issue_model_one(double *sink, cudaStream_t s)
{
    const int iters = 100, blocks = device_sms();
    cudaEvent_t a, b;
    cudaEventCreate(&a);
    cudaEventCreate(&b);
    issue_model_kernel<HOG><<<blocks, 512, 0, s>>>(sink, 2, 1e-8, 3);
    cudaEventRecord(a, s);
    issue_model_kernel<HOG><<<blocks, 512, 0, s>>>(sink, iters, 1e-8, 3);
    cudaEventRecord(b, s);
    cudaEventSynchronize(b);
    float ms = 0.f;
    cudaEventElapsedTime(&ms, a, b);
    cudaEventDestroy(a);
    cudaEventDestroy(b);
    return (double)blocks * 8 * 32 * iters * 64.0 * 2.0 * 4 / (ms * 1e-3);   // body-source interactions per second
}

}  // namespace bh

using namespace bh;

extern "C" {

// measured fp64 FMA rate in TFLOP/s (2 flops per FMA), best of three; 0 on success
int bhmb_fp64_peak(void *cuda_stream, double *tflops_host)
{
    cudaStream_t s = (cudaStream_t)cuda_stream;
    double *sink = nullptr;
    if (!tflops_host || cudaMalloc(&sink, 256) != cudaSuccess) return -1;
    const int iters = 1 << 16, blocks = device_sms() * 8, threads = 256;
    cudaEvent_t a, b;
    cudaEventCreate(&a);
    cudaEventCreate(&b);
    fp64_peak_kernel<<<blocks, threads, 0, s>>>(sink, 1 << 10, 1.0);   // warm-up
    float best = 1e30f;
    for (int rep = 0; rep < 3; ++rep) {
        cudaEventRecord(a, s);
        fp64_peak_kernel<<<blocks, threads, 0, s>>>(sink, iters, 1.0);
        cudaEventRecord(b, s);
        cudaEventSynchronize(b);
        float ms = 0.f;
        cudaEventElapsedTime(&ms, a, b);
        if (ms < best) best = ms;
    }
    cudaEventDestroy(a);
    cudaEventDestroy(b);
    cudaFree(sink);
    const double flops = 2.0 * 8.0 * (double)iters * (double)blocks * (double)threads;
    *tflops_host = flops / (best * 1e-3) / 1e12;
    return cudaGetLastError() == cudaSuccess ? 0 : -1;
}

// body-source interactions per second of the walk's evaluation loop: [0] alone on the sub-partition, [1] beside
// two warps running a dependent integer / shared-memory chain at low duty, [2] beside two warps issuing
// independent integer instructions at full rate
int bhmb_issue_model(void *cuda_stream, double out_host[3])
{
    cudaStream_t s = (cudaStream_t)cuda_stream;
    double *sink = nullptr;
    if (!out_host || cudaMalloc(&sink, 256) != cudaSuccess) return -1;
    out_host[0] = run_issue_model_one<0>(sink, s);
    out_host[1] = run_issue_model_one<1>(sink, s);
    out_host[2] = run_issue_model_one<2>(sink, s);
    cudaFree(sink);
    return cudaGetLastError() == cudaSuccess ? 0 : -1;
}

// out[0] = DFMA alone, out[1] = fp64 MMA alone (TFLOP/s, 2 flops per FMA), out[2] = time of both interleaved in
// one warp divided by the sum of the two times alone (1.0: they share a datapath; 0.5: they overlap fully)
int bhmb_fp64_mma(void *cuda_stream, double out_host[3])
{
    cudaStream_t s = (cudaStream_t)cuda_stream;
    double *sink = nullptr;
    if (!out_host || cudaMalloc(&sink, 256) != cudaSuccess) return -1;
    const int blocks = device_sms() * 8, iters = 4000;
    const double work = (double)blocks * 256 * iters;
    const float t0 = run_fp64_mma_one<0>(sink, blocks, iters, s), t1 = run_fp64_mma_one<1>(sink, blocks, iters, s),
                t2 = run_fp64_mma_one<2>(sink, blocks, iters, s);
    cudaFree(sink);
    out_host[0] = work * 16.0 / (t0 * 1e-3) / 1e12;     // 8 FMA per thread and iteration
    out_host[1] = work * 128.0 / (t1 * 1e-3) / 1e12;    // 8 MMAs of 8 x 8 x 4 FMA per warp and iteration
    out_host[2] = t2 / (t0 + t1);
    return cudaGetLastError() == cudaSuccess ? 0 : -1;
}

}  // extern "C"
