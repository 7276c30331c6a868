// bh_grid.cuh — barrier of a co-resident grid (cooperative launch), used by the one-kernel build of mid-size sets
// (bh_mid.cu) and by the one-kernel sort (bh_sort.cu).
#pragma once
#include "bh_common.cuh"

namespace bh {

// Barrier of the first `nblocks` blocks of the (co-resident) grid; bar[0] counts arrivals, bar[1] is the generation.
// Arrival is an acq_rel atomic (it publishes the block's writes and, for the last block, acquires everybody else's),
// the last block opens the barrier with a release, the others poll the generation with ld.acquire — on sm_100 an
// acquire load is LDG.STRONG.GPU + CCTL.IVALL, i.e. it also drops the SM's L1, which is what makes the plain loads
// of the next phase safe.
__device__ __forceinline__ void grid_barrier(unsigned *bar, unsigned nblocks)
{
    __syncthreads();
    if (threadIdx.x == 0) {
        unsigned gen, old;
        asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(gen) : "l"(bar + 1) : "memory");
        asm volatile("atom.acq_rel.gpu.global.add.u32 %0, [%1], 1;" : "=r"(old) : "l"(bar) : "memory");
        if (old == nblocks - 1u) {
            asm volatile("st.relaxed.gpu.global.u32 [%0], %1;" ::"l"(bar), "r"(0u) : "memory");
            asm volatile("red.release.gpu.global.add.u32 [%0], 1;" ::"l"(bar + 1) : "memory");
        }
        unsigned now;
        do {
            asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(now) : "l"(bar + 1) : "memory");
        } while (now == gen);
    }
    __syncthreads();
}

}  // namespace bh
