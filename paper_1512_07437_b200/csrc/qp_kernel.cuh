// qp_kernel.cuh -- the persistent pair kernel ("length-binned pair scheduler that packs many
// short pairs per CTA and splits long pairs across a CTA by anti-diagonal wavefront").
//   packed classes (W = 1): every warp owns one scratch slot and pulls pairs of its class largest-first;
//   split classes  (W > 1): every CTA owns one scratch slot, its W warps share each pair it pulls.
#pragma once
#include "qp_pair.cuh"

namespace qp {

template <typename R, int C, int W> struct KernelSmem {
    using V2 = typename Traits<R>::vec2;
    static constexpr int kWarps = W == 1 ? kWarpsPerCta : W;
    static constexpr size_t tab = sizeof(V2) * kTabDim * kTabDim;
    static constexpr size_t mbars = 256;   // kWarps * kStages mbarriers
    static constexpr size_t rings = (size_t)kWarps * RingBytes<R, C>::v + RingBytes<R, C>::stage;   // + one zeroed stage
    static_assert(kWarps * kStages * 8 <= (int)mbars, "mbarrier area");
    template <int GP> static constexpr size_t total() {
        return tab + mbars + rings + (W > 1 ? ((sizeof(CoopShared<R, GP, W>) + 127) & ~(size_t)127) : 0);
    }
};

template <typename R, int GP, int C, int MODE, int W>
__global__ void __launch_bounds__(KernelSmem<R, C, W>::kWarps * 32, ctas_per_sm(C, W, sizeof(R) == 8))
pair_kernel(const __grid_constant__ KArgs<R> ka) {
    using V2 = typename Traits<R>::vec2;
    using SM = KernelSmem<R, C, W>;
    constexpr int kWarps = SM::kWarps;
    // dynamic shared memory: emission table | kStages mbarriers per warp | F ring per warp | one zeroed stage | CoopShared
    extern __shared__ __align__(128) unsigned char smem_raw[];
    V2* tab = (V2*)smem_raw;
    uint64_t* mbars = (uint64_t*)(smem_raw + SM::tab);
    unsigned char* rings = smem_raw + SM::tab + SM::mbars;
    CoopShared<R, GP, W>* cs = (CoopShared<R, GP, W>*)(rings + SM::rings);   // only touched when W > 1
    for (int q = threadIdx.x; q < kTabDim * kTabDim; q += blockDim.x) tab[q] = ka.tab[q];
    for (int q = threadIdx.x; q < (int)(SM::rings / 16); q += blockDim.x) ((float4*)rings)[q] = make_float4(0.f, 0.f, 0.f, 0.f);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    FRing ring;
    ring.data = smem_u32(rings + warp * RingBytes<R, C>::v);
    ring.mbar = smem_u32(mbars + warp * kStages);
    ring.zeros = smem_u32(rings + kWarps * RingBytes<R, C>::v);
    ring.issued = ring.waited = 0;
    if (lane == 0) {
        for (int q = 0; q < kStages; ++q) mbar_init(ring.mbar + q * 8, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    fence_proxy_async();   // ring zeroing (generic proxy) before the first bulk copy lands in it
    __syncthreads();
    constexpr int cls = class_index(C, W, sizeof(R) == 8);
    const int unit = W == 1 ? blockIdx.x * kWarpsPerCta + warp : blockIdx.x;   // who owns a scratch slot
    SchedHeader* hdr = ka.hdr;
    int granted, count;
    const int32_t* list;
    char* slot;
    int* cursor;
    if (ka.refine_pass) {
        granted = hdr->refine_W[cls];
        count = hdr->refine_count[cls];
        list = ka.refine_list + (int64_t)cls * ka.refine_stride;
        if (unit >= granted) return;
        slot = ka.slots + hdr->refine_slot0[cls] + (unsigned long long)unit * hdr->refine_slot_bytes[cls];
        cursor = &hdr->refine_cursor[cls];
    } else {
        granted = hdr->cls_W[cls];
        count = hdr->cls_count[cls];
        list = ka.order + hdr->cls_start[cls];
        if (unit >= granted) return;
        slot = ka.slots + ka.slot_off[hdr->cls_slot0[cls] + unit];
        cursor = &hdr->cls_cursor[cls];
    }
    int idx = unit;   // the first `granted` pairs of the (largest-first) list go to units 0..granted-1; the rest are pulled
    while (idx < count) {
        process_pair<R, GP, C, MODE, W>(ka, smem_u32(tab), list[idx], slot, lane, warp, ring, cs);
        if constexpr (W == 1) {
            if (lane == 0) idx = atomicAdd(cursor, 1);
            idx = __shfl_sync(kFull, idx, 0);
        } else {
            cta_sync();   // every warp is done with the slot and with CoopShared
            if (threadIdx.x == 0) cs->next = atomicAdd(cursor, 1);
            cta_sync();
            idx = cs->next;
        }
    }
}

template <typename R, int GP, int C, int MODE, int W> cudaError_t launch_pair(const KArgs<R>& ka, int grid, cudaStream_t st) {
    constexpr size_t smem = KernelSmem<R, C, W>::template total<GP>();
    static bool attr_set = false;   // per instantiation; the attribute is sticky per device function
    if (!attr_set) {
        cudaError_t e = cudaFuncSetAttribute(pair_kernel<R, GP, C, MODE, W>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        attr_set = true;
    }
    pair_kernel<R, GP, C, MODE, W><<<grid, KernelSmem<R, C, W>::kWarps * 32, smem, st>>>(ka);
    return cudaGetLastError();
}

}  // namespace qp
