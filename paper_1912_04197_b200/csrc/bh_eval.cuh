// bh_eval.cuh — the fp64 interaction arithmetic of the walk (a7) and direct (a8) kernels: Eqs. (4)-(6)
// PAPER.md:90-101 per body-source pair, and the consumer's evaluation loop over a shared-memory ring of
// sources.  Shared by bh_walk.cu and the measurement-only microbenchmarks (csrc/bench/), which time this very
// loop; nothing here is shared with oracle/.
#pragma once
#include "bh_common.cuh"

namespace bh {

constexpr int kRing = 512;                  // sources per producer/consumer pair (power of two, multiple of 8)
// GUARD (chosen by the launchers when eps^2 is below the smallest normal double, eps = 0 included): a softened
// squared distance that is zero or subnormal adds nothing.  rsqrt.approx.ftz flushes a subnormal argument to
// zero and would return infinity, and with it 0 * inf = NaN for a coincident pair (R13; bh.h preconditions).
constexpr double kTinyR2 = 2.2250738585072014e-308;

// m / r^3 from r2 = |d|^2 + eps^2: MUFU.RSQ64H seed y (about 20 good bits), e = 1 - r2 y^2 and the
// series (1-e)^(-3/2) = 1 + e (3/2 + 15/8 e) + O(e^3).  Every fp64 instruction except the three
// accumulations reads at most two distinct register operands (a third costs the pipe a cycle on sm_100).
template <bool GUARD>
__device__ __forceinline__ void interact(double px, double py, double pz, double eps2, const double4 s,
                                         double &ax, double &ay, double &az)
{
    const double dx = s.x - px, dy = s.y - py, dz = s.z - pz;
    const double t2 = fma(dy, dy, fma(dz, dz, eps2));
    const double r2 = fma(dx, dx, t2);
    double y;
    // the seed's low word is irrelevant (the series below corrects any y within 2^-19 of r2^-1/2): take it
    // from the dead partial sum, so that MUFU.RSQ64H can write into that register pair without a zero-fill
    {
        double y0;
        asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y0) : "d"(r2));
        y = __hiloint2double(__double2hiint(y0), __double2loint(t2));
    }
    if (GUARD) y = (r2 >= kTinyR2) ? y : 0.0;  // a pair at zero softened distance adds nothing (R13)
    const double u = y * y;
    const double w = s.w * y;
    const double e = fma(-r2, u, 1.0);
    const double v = u * w;
    const double p = fma(1.875, e, 1.5);
    const double h = fma(p, e, 1.0);
    const double f = v * h;
    ax = fma(f, dx, ax);
    ay = fma(f, dy, ay);
    az = fma(f, dz, az);
}

// m / r from the same seed (NEXT-1, potential of the softened force, R24): (1-e)^(-1/2) = 1 + e (1/2 + 3/8 e) + O(e^3)
template <bool GUARD>
__device__ __forceinline__ void interact_pot(double px, double py, double pz, double eps2, const double4 s, double &phi)
{
    const double dx = s.x - px, dy = s.y - py, dz = s.z - pz;
    const double r2 = fma(dx, dx, fma(dy, dy, fma(dz, dz, eps2)));
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(r2));
    if (GUARD) y = (r2 >= kTinyR2) ? y : 0.0;
    const double u = y * y;
    const double w = s.w * y;
    const double e = fma(-r2, u, 1.0);
    const double p = fma(0.375, e, 0.5);
    const double h = fma(p, e, 1.0);
    phi = fma(w, h, phi);
}

// acceleration and potential of one interaction from one seed: 16 + 3 fp64 instructions
template <bool GUARD>
__device__ __forceinline__ void interact_both(double px, double py, double pz, double eps2, const double4 s,
                                              double &ax, double &ay, double &az, double &phi)
{
    const double dx = s.x - px, dy = s.y - py, dz = s.z - pz;
    const double t2 = fma(dy, dy, fma(dz, dz, eps2));
    const double r2 = fma(dx, dx, t2);
    double y;
    {
        double y0;
        asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y0) : "d"(r2));
        y = __hiloint2double(__double2hiint(y0), __double2loint(t2));
    }
    if (GUARD) y = (r2 >= kTinyR2) ? y : 0.0;
    const double u = y * y;
    const double w = s.w * y;
    const double e = fma(-r2, u, 1.0);
    const double v = u * w;
    const double p = fma(1.875, e, 1.5);
    const double q = fma(0.375, e, 0.5);
    const double h = fma(p, e, 1.0);
    const double g = fma(q, e, 1.0);
    const double f = v * h;
    phi = fma(w, g, phi);
    ax = fma(f, dx, ax);
    ay = fma(f, dy, ay);
    az = fma(f, dz, az);
}

// MODE 0: accelerations, 1: potential (accumulated in ax), 2: both
template <bool GUARD, int MODE>
__device__ __forceinline__ void interact_any(double px, double py, double pz, double eps2, const double4 s,
                                             double &ax, double &ay, double &az, double &ph)
{
    if constexpr (MODE == 1) interact_pot<GUARD>(px, py, pz, eps2, s, ax);
    else if constexpr (MODE == 2) interact_both<GUARD>(px, py, pz, eps2, s, ax, ay, az, ph);
    else interact<GUARD>(px, py, pz, eps2, s, ax, ay, az);
}

// Lane l = 8 q + r holds bodies r, r+8, r+16, r+24 of the group (NS = ceil(bodies / 8) of them are
// real) and, of every chunk of eight sources, takes sources q and q+4.
template <int NS>
struct Bodies {
    double x[NS], y[NS], z[NS], ax[NS], ay[NS], az[NS], ph[NS];   // ph only lives in MODE 2
};

// evaluate n8 (a multiple of 8) sources starting at ring position head (a multiple of 8): the end of a list
template <bool GUARD, int NS, int MODE>
__device__ __forceinline__ void eval_chunks(const double4 *ring, unsigned head, unsigned n8, unsigned quarter,
                                            double eps2, Bodies<NS> &B)
{
#pragma unroll 1
    for (unsigned i = 0; i < n8; i += 8) {
        const double4 *p = ring + ((head + i) & (kRing - 1)) + quarter;
        const double4 s0 = p[0], s1 = p[4];
#pragma unroll
        for (int k = 0; k < NS; ++k) interact_any<GUARD, MODE>(B.x[k], B.y[k], B.z[k], eps2, s0, B.ax[k], B.ay[k], B.az[k], B.ph[k]);
#pragma unroll
        for (int k = 0; k < NS; ++k) interact_any<GUARD, MODE>(B.x[k], B.y[k], B.z[k], eps2, s1, B.ax[k], B.ay[k], B.az[k], B.ph[k]);
    }
}

// the same over n32 (a multiple of 32) sources starting at a ring position that is a multiple of 32: a block of
// four chunks never wraps, so it has ONE ring address and constant offsets (the chunk-wise loop computes a masked
// address per chunk: 13 more integer instructions per 512 fp64 ones, and every one of them takes an issue slot)
template <bool GUARD, int NS, int MODE>
__device__ __forceinline__ void eval_blocks(const double4 *ring, unsigned head, unsigned n32, unsigned quarter,
                                            double eps2, Bodies<NS> &B)
{
    // the first two sources of the NEXT block are requested while the last chunk of this one is evaluated, so a
    // block does not start with an exposed shared-memory latency
    if (n32 == 0) return;
    const double4 *p = ring + (head & (kRing - 1)) + quarter;
    double4 s0 = p[0], s1 = p[4];
#pragma unroll 1
    for (unsigned i = 0; i < n32; i += 32) {
        // (after the last block of the batch the request goes to this block again: nothing beyond the published limit is read)
        const double4 *pn = ring + ((head + (i + 32 < n32 ? i + 32 : i)) & (kRing - 1)) + quarter;
#pragma unroll
        for (int c = 0; c < 4; ++c) {
            const double4 a0 = s0, a1 = s1;
            if (c < 3) { s0 = p[8 * c + 8]; s1 = p[8 * c + 12]; }
            else { s0 = pn[0]; s1 = pn[4]; }
#pragma unroll
            for (int k = 0; k < NS; ++k) interact_any<GUARD, MODE>(B.x[k], B.y[k], B.z[k], eps2, a0, B.ax[k], B.ay[k], B.az[k], B.ph[k]);
#pragma unroll
            for (int k = 0; k < NS; ++k) interact_any<GUARD, MODE>(B.x[k], B.y[k], B.z[k], eps2, a1, B.ax[k], B.ay[k], B.az[k], B.ph[k]);
        }
        p = pn;
    }
}

}  // namespace bh
