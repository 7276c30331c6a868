// bh_sort.cuh — block-level pieces of step a3 shared by the onesweep passes (bh_sort.cu) and the one-block
// build of small body sets (bh_small.cu): a 256-thread exclusive scan and a stable LSD radix sort of up to
// 256 x ITEMS (key, index) pairs that never leaves registers and shared memory.
#pragma once
#include "bh_common.cuh"

namespace bh {

// exclusive scan of one value per thread over a 256-thread block; tmp is 8 words of shared memory
__device__ __forceinline__ unsigned block_excl_scan_256(unsigned v, unsigned *tmp)
{
    const unsigned lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
    unsigned inc = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        unsigned t = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= (unsigned)o) inc += t;
    }
    if (lane == 31) tmp[warp] = inc;
    __syncthreads();
    unsigned base = 0;
#pragma unroll
    for (int k = 0; k < 8; ++k)
        if ((unsigned)k < warp) base += tmp[k];
    __syncthreads();
    return base + inc - v;
}

// exclusive scan of one value per digit (threads 0..255 hold a digit each, the others pass 0) over a block of
// THREADS >= 256 threads; tmp is 8 words of shared memory
template <int THREADS>
__device__ __forceinline__ unsigned block_excl_scan_digits(unsigned v, unsigned *tmp)
{
    const unsigned lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
    unsigned inc = v;
    if (warp < 8) {
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            unsigned t = __shfl_up_sync(0xffffffffu, inc, o);
            if (lane >= (unsigned)o) inc += t;
        }
        if (lane == 31) tmp[warp] = inc;
    }
    __syncthreads();
    unsigned base = 0;
#pragma unroll
    for (int k = 0; k < 8; ++k)
        if ((unsigned)k < warp) base += tmp[k];
    __syncthreads();
    return base + inc - v;
}

// Lanes of the warp that carry the same digit as this lane, from one ballot per digit bit (valid lanes only; an
// invalid lane is alone).  match.any gives the same mask in one instruction, but on sm_100 the eight ballots are
// much the faster way: the sort passes took 171 -> 134 us at 1M keys and 455 -> 359 us at 4M with them (measured,
// round 2), and the ncu capture of the match.any version had half of a pass's stall samples on the instruction
// after the match.
__device__ __forceinline__ unsigned digit_peers(unsigned d, bool valid, unsigned lane)
{
    unsigned peers = __ballot_sync(0xffffffffu, valid);
#pragma unroll
    for (int b = 0; b < kRadixBits; ++b) {
        const bool bit = (d >> b) & 1u;
        const unsigned m = __ballot_sync(0xffffffffu, bit);
        peers &= bit ? m : ~m;
    }
    return valid ? peers : (1u << lane);
}

// Rank of a key among the keys of its warp that carry the same digit and came before it (earlier rows, then lower
// lanes: index order, so the sort is stable).  cnt[256] are the warp's own running digit counters.
__device__ __forceinline__ unsigned warp_rank(unsigned *cnt, unsigned d, bool valid, unsigned lane, unsigned lt)
{
    const unsigned peers = digit_peers(d, valid, lane);
    const unsigned pre = valid ? cnt[d] : 0u;
    __syncwarp();
    if (valid && (peers & lt) == 0u) cnt[d] = pre + __popc(peers);
    __syncwarp();
    return pre + __popc(peers & lt);
}

// All eight digit passes inside one block of THREADS threads (a step over a few thousand bodies is bound by the
// latency of its dependent launches, "for a low number of bodies the computational time is dominated
// by the octree creation").  Thread t holds items  idx = warp * 32 * ITEMS + i * 32 + lane  (i < ITEMS), before and
// after; padding keys ~0 sort last in every pass (all digits 255, after the real 255s: stable).  Per-warp
// ballot ranking as in the tiled passes: stable by construction (item order, then lane order = index order).
// skey: THREADS * ITEMS keys of shared memory (reused for the values); whist: [THREADS / 32][256]; stoff: [256];
// stmp: [8].
template <int ITEMS, int THREADS>
__device__ __forceinline__ void block_radix_sort(unsigned long long (&k)[ITEMS], unsigned (&v)[ITEMS],
                                                 unsigned long long *skey, unsigned (*whist)[kRadix], unsigned *stoff,
                                                 unsigned *stmp)
{
    constexpr int kWarps = THREADS / 32;
    const unsigned tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
    const unsigned lt = (1u << lane) - 1u;
    unsigned pos[ITEMS];
#pragma unroll 1
    for (int p = 0; p < kSortPasses; ++p) {
        const int shift = p * kRadixBits;
        for (int q = tid; q < kWarps * kRadix; q += THREADS) (&whist[0][0])[q] = 0u;
        __syncthreads();
#pragma unroll
        for (int i = 0; i < ITEMS; ++i) {
            const unsigned d = (unsigned)(k[i] >> shift) & (kRadix - 1);
            pos[i] = warp_rank(whist[warp], d, true, lane, lt);
        }
        __syncthreads();
        unsigned tot = 0;
        if (tid < (unsigned)kRadix) {   // digit = tid: exclusive prefix over the warps, total
#pragma unroll 8
            for (int w = 0; w < kWarps; ++w) {
                const unsigned c = whist[w][tid];
                whist[w][tid] = tot;
                tot += c;
            }
        }
        const unsigned off = block_excl_scan_digits<THREADS>(tot, stmp);
        if (tid < (unsigned)kRadix) stoff[tid] = off;
        __syncthreads();
#pragma unroll
        for (int i = 0; i < ITEMS; ++i) {
            const unsigned d = (unsigned)(k[i] >> shift) & (kRadix - 1);
            pos[i] += stoff[d] + whist[warp][d];
            skey[pos[i]] = k[i];
        }
        __syncthreads();
#pragma unroll
        for (int i = 0; i < ITEMS; ++i) k[i] = skey[warp * (32 * ITEMS) + i * 32 + lane];
        __syncthreads();
        unsigned *sval = reinterpret_cast<unsigned *>(skey);
#pragma unroll
        for (int i = 0; i < ITEMS; ++i) sval[pos[i]] = v[i];
        __syncthreads();
#pragma unroll
        for (int i = 0; i < ITEMS; ++i) v[i] = sval[warp * (32 * ITEMS) + i * 32 + lane];
        __syncthreads();
    }
}

}  // namespace bh
