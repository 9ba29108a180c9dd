// qp_kernel.cuh -- the persistent pair kernel: every warp owns one scratch slot and pulls pairs of its
// scheduling class longest-first from a device-side queue ("length-binned pair scheduler").
#pragma once
#include "qp_pair.cuh"

namespace qp {

template <typename R, int GP, int C, int MODE>
__global__ void __launch_bounds__(kWarpsPerCta * 32, ctas_per_sm(C, sizeof(R) == 8))
pair_kernel(const __grid_constant__ KArgs<R> ka) {
    using V2 = typename Traits<R>::vec2;
    // dynamic shared memory: emission table | kStages mbarriers per warp | F ring per warp | one zeroed stage (FRing)
    extern __shared__ __align__(128) unsigned char smem_raw[];
    V2* tab = (V2*)smem_raw;
    uint64_t* mbars = (uint64_t*)(smem_raw + sizeof(V2) * kTabDim * kTabDim);
    unsigned char* rings = smem_raw + sizeof(V2) * kTabDim * kTabDim + 128;
    static_assert(kWarpsPerCta * kStages * 8 <= 128, "mbarrier area");
    for (int q = threadIdx.x; q < kTabDim * kTabDim; q += blockDim.x) tab[q] = ka.tab[q];
    for (int q = threadIdx.x; q < (kWarpsPerCta * RingBytes<R, C>::v + RingBytes<R, C>::stage) / 16; q += blockDim.x)
        ((float4*)rings)[q] = make_float4(0.f, 0.f, 0.f, 0.f);
    FRing ring;
    ring.data = smem_u32(rings + (threadIdx.x >> 5) * RingBytes<R, C>::v);
    ring.mbar = smem_u32(mbars + (threadIdx.x >> 5) * kStages);
    ring.zeros = smem_u32(rings + kWarpsPerCta * RingBytes<R, C>::v);
    ring.issued = ring.waited = 0;
    if ((threadIdx.x & 31) == 0) {
        for (int q = 0; q < kStages; ++q) mbar_init(ring.mbar + q * 8, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    fence_proxy_async();   // ring zeroing (generic proxy) before the first bulk copy lands in it
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
        process_pair<R, GP, C, MODE>(ka, tab, list[idx], slot, lane, ring);
        if (lane == 0) idx = atomicAdd(cursor, 1);
        idx = __shfl_sync(kFull, idx, 0);
    }
}

template <typename R, int C> constexpr size_t pair_smem_bytes() {
    return sizeof(typename Traits<R>::vec2) * kTabDim * kTabDim + 128 + (size_t)kWarpsPerCta * RingBytes<R, C>::v + RingBytes<R, C>::stage;
}

template <typename R, int GP, int C, int MODE> cudaError_t launch_pair(const KArgs<R>& ka, int grid, cudaStream_t st) {
    constexpr size_t smem = pair_smem_bytes<R, C>();
    static bool attr_set = false;   // per instantiation; the attribute is sticky per device function
    if (!attr_set) {
        cudaError_t e = cudaFuncSetAttribute(pair_kernel<R, GP, C, MODE>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        attr_set = true;
    }
    pair_kernel<R, GP, C, MODE><<<grid, kWarpsPerCta * 32, smem, st>>>(ka);
    return cudaGetLastError();
}

}  // namespace qp
