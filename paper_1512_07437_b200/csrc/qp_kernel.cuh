// qp_kernel.cuh -- the persistent pair kernel: every warp owns one scratch slot and pulls pairs of its
// scheduling class longest-first from a device-side queue ("length-binned pair scheduler").
#pragma once
#include "qp_pair.cuh"

namespace qp {

template <typename R, int GP, int C, int MODE>
__global__ void __launch_bounds__(kWarpsPerCta * 32, ctas_per_sm(C, sizeof(R) == 8))
pair_kernel(const __grid_constant__ KArgs<R> ka) {
    using V2 = typename Traits<R>::vec2;
    __shared__ V2 tab[kTabDim * kTabDim];
    for (int q = threadIdx.x; q < kTabDim * kTabDim; q += blockDim.x) tab[q] = ka.tab[q];
    __syncthreads();
    constexpr int cls = C / 2 - 1;
    const int lane = threadIdx.x & 31;
    const int gw = blockIdx.x * kWarpsPerCta + (threadIdx.x >> 5);
    SchedHeader* hdr = ka.hdr;
    int W, count;
    const int32_t* list;
    char* slot;
    int* cursor;
    if (ka.refine_pass) {
        W = hdr->refine_W[cls];
        count = hdr->refine_count[cls];
        list = ka.refine_list + (int64_t)cls * ka.refine_stride;
        if (gw >= W) return;
        slot = ka.slots + hdr->refine_slot0[cls] + (unsigned long long)gw * hdr->refine_slot_bytes[cls];
        cursor = &hdr->refine_cursor[cls];
    } else {
        W = hdr->cls_W[cls];
        count = hdr->cls_count[cls];
        list = ka.order + hdr->cls_start[cls];
        if (gw >= W) return;
        slot = ka.slots + ka.slot_off[hdr->cls_slot0[cls] + gw];
        cursor = &hdr->cls_cursor[cls];
    }
    int idx = gw;   // the first W pairs of the (largest-first) list go to warps 0..W-1; the rest are pulled
    while (idx < count) {
        process_pair<R, GP, C, MODE>(ka, tab, list[idx], slot, lane);
        if (lane == 0) idx = atomicAdd(cursor, 1);
        idx = __shfl_sync(kFull, idx, 0);
    }
}

template <typename R, int GP, int C, int MODE> cudaError_t launch_pair(const KArgs<R>& ka, int grid, cudaStream_t st) {
    pair_kernel<R, GP, C, MODE><<<grid, kWarpsPerCta * 32, 0, st>>>(ka);
    return cudaGetLastError();
}

}  // namespace qp
