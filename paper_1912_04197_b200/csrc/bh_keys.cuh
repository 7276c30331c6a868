// bh_keys.cuh — device helpers of steps a1 / a2 shared by the streaming kernels (bh_keys.cu) and the
// one-block build of small body sets (bh_small.cu): canonical cube from the per-axis extremes (R11),
// quantisation and Morton interleave (R12).
#pragma once
#include "bh_common.cuh"

namespace bh {

__device__ __forceinline__ bool nonfinite(double x)
{
    return (__double2hiint(x) & 0x7ff00000) == 0x7ff00000;
}

// Derive the cube from the per-axis minima / maxima (R11: corner = per-axis minimum, side = smallest power of
// two strictly above the largest extent, 1 if the extent is 0), flag non-finite input and an extent outside the
// documented range, and reset the per-build words of the device state.  One thread.
__device__ __forceinline__ void finish_cube(double lo[3], const double hi[3], int bad, DevState *st)
{
    double E = 0.0;
    for (int a = 0; a < 3; ++a) E = fmax(E, __dsub_rn(hi[a], lo[a]));   // one rounding per extent
    if (nonfinite(E)) bad = 1;
    int e = 0;
    if (bad) {   // keep every later kernel memory-safe; the error is reported by the host
        lo[0] = lo[1] = lo[2] = 0.0;
    } else if (E != 0.0) {
        (void)frexp(E, &e);   // E = f 2^e, 1/2 <= f < 1  =>  2^(e-1) <= E < 2^e
    }
    st->lo[0] = lo[0];
    st->lo[1] = lo[1];
    st->lo[2] = lo[2];
    st->e = e;
    st->side = ldexp(1.0, e);
    st->scale = ldexp(1.0, 21 - e);
    // sticky error bits: OR-ed in, cleared by the host once it has reported them (bh.h)
    int flags = bad ? (int)kStatNonFinite : 0;
    if (!bad && E != 0.0 && (e < -kMaxExtentExp + 1 || e > kMaxExtentExp + 1)) flags |= (int)kStatRange;
    if (flags) atomicOr(&st->status, flags);
    st->n_nodes = 0;
    st->n_groups = 0;
    st->depth = 0;
    st->ticket_bbox = 0;
    st->walk_queue = 0;
    st->walk_done = 0;
    for (int k = 0; k < kNumStats; ++k) st->stats[k] = 0ull;
}

// spread the low 21 bits of v so that bit k lands on bit 3k
__device__ __forceinline__ unsigned long long spread3(unsigned v)
{
    unsigned long long x = v & 0x1fffffu;
    x = (x | (x << 32)) & 0x001f00000000ffffull;
    x = (x | (x << 16)) & 0x001f0000ff0000ffull;
    x = (x | (x << 8)) & 0x100f00f00f00f00full;
    x = (x | (x << 4)) & 0x10c30c30c30c30c3ull;
    x = (x | (x << 2)) & 0x1249249249249249ull;
    return x;
}

__device__ __forceinline__ unsigned quantise(double x, double lo, double scale)
{
    // one rounded subtraction, exact power-of-two scaling, truncation (R11/R12); the clamp is a
    // no-op for finite input (x - lo <= extent < L) and keeps non-finite input memory-safe
    double d = __dmul_rn(__dsub_rn(x, lo), scale);
    d = fmin(fmax(d, 0.0), 2097151.0);
    return (unsigned)__double2uint_rz(d);
}

__device__ __forceinline__ unsigned long long morton_key(double x, double y, double z, double lx, double ly, double lz,
                                                         double sc)
{
    return spread3(quantise(x, lx, sc)) | (spread3(quantise(y, ly, sc)) << 1) | (spread3(quantise(z, lz, sc)) << 2);
}

}  // namespace bh
