// sph_active.cu -- the active set of a rung: "only the particles on the
// active rungs are updated".  sph_set_active turns a per-particle mask (caller order) into the
// ascending list of the sorted positions of the active particles; the density and force
// sweeps then take their targets from that list (sources are always all particles).
// Ordered stream compaction in three launches over SPH_SCAN_BLOCKS fixed segments:
// count per segment, exclusive scan of the counts, ordered write.
#include <cstdio>
#include "sph_internal.cuh"

namespace {

constexpr int A_TPB = 256;

// flags in sorted order (rank is build-time scratch)
__global__ void k_act_flags(int64_t n, const int32_t* __restrict__ inv_perm,
                            const uint8_t* __restrict__ active, uint32_t* flag_sorted) {
    int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i < n) flag_sorted[inv_perm[i]] = active[i] ? 1u : 0u;
}

__global__ __launch_bounds__(A_TPB) void k_act_count(int64_t n, int64_t seg,
                                                     const uint32_t* __restrict__ flag,
                                                     uint32_t* part) {
    __shared__ unsigned sh;
    if (threadIdx.x == 0) sh = 0u;
    __syncthreads();
    const int64_t lo = blockIdx.x * seg, hi = min(n, lo + seg);
    unsigned      c  = 0;
    for (int64_t p = lo + threadIdx.x; p < hi; p += A_TPB) c += flag[p];
    c = __reduce_add_sync(SPH_FULL, c);
    if ((threadIdx.x & 31) == 0 && c) atomicAdd(&sh, c);
    __syncthreads();
    if (threadIdx.x == 0) part[blockIdx.x] = sh;
}

// exclusive scan of the SPH_SCAN_BLOCKS segment counts by one block; the total is the length
__global__ __launch_bounds__(SPH_SCAN_BLOCKS) void k_act_scan(uint32_t* part, unsigned* act_cnt) {
    __shared__ unsigned wsum[32];
    const int      t = threadIdx.x, lane = t & 31, w = t >> 5;
    const unsigned v = part[t];
    unsigned       x = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const unsigned y = __shfl_up_sync(SPH_FULL, x, o);
        if (lane >= o) x += y;
    }
    if (lane == 31) wsum[w] = x;
    __syncthreads();
    if (w == 0) {
        unsigned s = wsum[lane];
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const unsigned y = __shfl_up_sync(SPH_FULL, s, o);
            if (lane >= o) s += y;
        }
        wsum[lane] = s;   // inclusive over the warps
    }
    __syncthreads();
    const unsigned base = w ? wsum[w - 1] : 0u;
    part[t] = base + x - v;
    if (t == SPH_SCAN_BLOCKS - 1) *act_cnt = base + x;
}

__global__ __launch_bounds__(A_TPB) void k_act_write(int64_t n, int64_t seg,
                                                     const uint32_t* __restrict__ flag,
                                                     const uint32_t* __restrict__ part,
                                                     uint32_t* act_list) {
    __shared__ unsigned wcnt[A_TPB / 32];
    const int64_t lo = blockIdx.x * seg, hi = min(n, lo + seg);
    const int     lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    unsigned      base = part[blockIdx.x];
    for (int64_t p0 = lo; p0 < hi; p0 += A_TPB) {
        const int64_t  p = p0 + threadIdx.x;
        const bool     f = p < hi && flag[p] != 0u;
        const unsigned b = __ballot_sync(SPH_FULL, f);
        if (lane == 0) wcnt[w] = __popc(b);
        __syncthreads();
        unsigned before = 0, total = 0;
#pragma unroll
        for (int k = 0; k < A_TPB / 32; ++k) {
            const unsigned ck = wcnt[k];
            if (k < w) before += ck;
            total += ck;
        }
        if (f) act_list[base + before + __popc(b & ((1u << lane) - 1u))] = (uint32_t)p;
        base += total;
        __syncthreads();
    }
}

}  // namespace

// mask (n bytes, caller order) -> ascending list of sorted positions + its length
int sph_launch_compact(sph_ctx* c, const uint8_t* mask, uint32_t* list, unsigned* cnt) {
    cudaStream_t  s = c->stream;
    const int64_t n = c->n;
    const int64_t seg = (n + SPH_SCAN_BLOCKS - 1) / SPH_SCAN_BLOCKS;
    uint32_t*     flag = c->rank;
    k_act_flags<<<(int)((n + 255) / 256), 256, 0, s>>>(n, c->inv_perm, mask, flag);
    k_act_count<<<SPH_SCAN_BLOCKS, A_TPB, 0, s>>>(n, seg, flag, c->scan_part);
    k_act_scan<<<1, SPH_SCAN_BLOCKS, 0, s>>>(c->scan_part, cnt);
    k_act_write<<<SPH_SCAN_BLOCKS, A_TPB, 0, s>>>(n, seg, flag, c->scan_part, list);
    SPH_CUDA_CHECK(c, cudaGetLastError());
    return SPH_OK;
}

int sph_launch_set_active(sph_ctx* c, const uint8_t* active) {
    return sph_launch_compact(c, active, c->act_list, c->act_cnt);
}
