// common.cuh -- shared device helpers of the RefDef CUDA path (sm_100a).
// No arithmetic of the method lives here: reductions, the grid barrier, load helpers.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#define RD_WARP 32
#define RD_SLICE 32          // sliced-ELL slice height = one warp
#define RD_CG_THREADS 1024   // persistent Algorithm-1 kernel: one CTA of 32 warps per SM
#define RD_MAX_K 64

namespace rd {

__device__ __forceinline__ double warp_sum(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
__device__ __forceinline__ double warp_max(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
}
__device__ __forceinline__ double warp_min(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fmin(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
}

// Block-wide sum in a fixed order (warp butterflies, then warp 0 over the warp results): the value is
// the same on every run for a given block size.  scratch: >= 32 doubles of shared memory.  Returns the sum
// in every thread.  Contains two __syncthreads().
__device__ __forceinline__ double block_sum(double v, double* scratch)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
    v = warp_sum(v);
    __syncthreads();  // scratch may still be read from a previous call
    if (lane == 0) scratch[warp] = v;
    __syncthreads();
    double s = (lane < nw) ? scratch[lane] : 0.0;
    return warp_sum(s);
}

// Streaming read of data that no kernel in flight writes (matrix values, indices, W, HW, m, d):
// non-coherent path, no L1 allocation pressure from the compiler's point of view.
__device__ __forceinline__ double ldg_f64(const double* p) { return __ldg(p); }
__device__ __forceinline__ int ldg_i32(const int32_t* p) { return __ldg(p); }

// ---- grid barrier for the persistent cooperative kernel -----------------------------------------------
// Classic counter + generation barrier.  Every CTA of the (co-resident, cooperatively launched) grid calls
// it the same number of times.  All global writes made by the CTA before the call are visible to every
// thread of every CTA after it: bar.sync orders the CTA's writes before thread 0's gpu-scope fence and
// release; the spinning thread acquires at gpu scope (which also invalidates this SM's L1) and the closing
// bar.sync hands that to the rest of the CTA.
struct GridBarrier {
    unsigned int count;
    unsigned int gen;
};

__device__ __forceinline__ unsigned int ld_acquire_u32(const unsigned int* p)
{
    unsigned int v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ unsigned int ld_relaxed_u32(const unsigned int* p)
{
    unsigned int v;
    asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_release_u32(unsigned int* p, unsigned int v)
{
    asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
__device__ __forceinline__ unsigned int atom_add_acqrel_u32(unsigned int* p, unsigned int v)
{
    unsigned int old;
    asm volatile("atom.acq_rel.gpu.global.add.u32 %0, [%1], %2;" : "=r"(old) : "l"(p), "r"(v) : "memory");
    return old;
}

// Single-hop variant: one monotone 64-bit arrival counter; CTA number `gen` (1, 2, ...) of this launch is through
// when the counter reaches gen * nblocks.  Arrival is a release reduction without a return value (no round trip),
// everybody polls the counter itself with acquire loads: one L2 round trip after the last arrival instead of
// fence + atomic + reset + fence + release-store + poll.  The counter must be zero at launch.
__device__ __forceinline__ void grid_barrier_counter(unsigned long long* counter, unsigned int nblocks, unsigned int gen)
{
    __syncthreads();
    if (threadIdx.x == 0) {
        const unsigned long long target = (unsigned long long)gen * nblocks;
        asm volatile("red.release.gpu.global.add.u64 [%0], %1;" ::"l"(counter), "l"(1ull) : "memory");
        unsigned long long seen;
        do {
            asm volatile("ld.acquire.gpu.global.u64 %0, [%1];" : "=l"(seen) : "l"(counter) : "memory");
        } while (seen < target);
    }
    __syncthreads();
}

__device__ __forceinline__ void grid_barrier(GridBarrier* bar, unsigned int nblocks)
{
    __syncthreads();
    if (threadIdx.x == 0) {
        const unsigned int g = ld_acquire_u32(&bar->gen);
        __threadfence();
        const unsigned int arrived = atom_add_acqrel_u32(&bar->count, 1u);
        if (arrived == nblocks - 1) {
            bar->count = 0;  // nobody touches count again before observing the new generation
            __threadfence();
            st_release_u32(&bar->gen, g + 1);
        } else {
            while (ld_acquire_u32(&bar->gen) == g) { __nanosleep(20); }
        }
        __threadfence();
    }
    __syncthreads();
}

}  // namespace rd
