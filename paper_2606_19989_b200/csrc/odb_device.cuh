// Device-side helpers shared by the kernels of libodb (CUDA path only): warp / block scans, stream
// compaction, acquire / release flag accesses.
#pragma once

#include "odb_internal.cuh"

namespace odb {

template <class V>
__device__ __forceinline__ V warp_incl_scan(V v) {
    const int lane = threadIdx.x & 31;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        V n = __shfl_up_sync(ODB_FULL_MASK, v, d);
        if (lane >= d) v += n;
    }
    return v;
}

// Exclusive scan of one value per thread over the CTA.  `s` is shared scratch of 34 V's.
// Returns the exclusive prefix; `total` receives the CTA-wide sum.  Contains barriers: every
// thread of the CTA must call it.
template <class V>
__device__ __forceinline__ V block_excl_scan(V v, V *s, V &total) {
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
    V inc = warp_incl_scan(v);
    if (lane == 31) s[w] = inc;
    __syncthreads();
    if (w == 0) {
        V x = lane < nw ? s[lane] : (V)0;
        V xi = warp_incl_scan(x);
        s[lane] = xi - x;
        if (lane == 31) s[32] = xi;
    }
    __syncthreads();
    V r = inc - v + s[w];
    total = s[32];
    __syncthreads();
    return r;
}

// Stream compaction over i in [0, n): emit(i, k) for the k-th i with pred(i).  Returns the count.
template <class Pred, class Emit>
__device__ __forceinline__ int block_compact(int n, int *s, Pred pred, Emit emit) {
    int carry = 0;
    for (int base = 0; base < n; base += blockDim.x) {
        int i = base + threadIdx.x;
        int f = (i < n && pred(i)) ? 1 : 0;
        int tot;
        int ex = block_excl_scan<int>(f, s, tot);
        if (f) emit(i, carry + ex);
        carry += tot;
    }
    return carry;
}

__device__ __forceinline__ int ld_flag(const int *p) {
    int v;
    asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_flag(int *p, int v) {
    asm volatile("st.release.gpu.global.s32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}


}  // namespace odb
