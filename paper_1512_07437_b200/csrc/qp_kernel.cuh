// qp_kernel.cuh -- the persistent pair kernel ("length-binned pair scheduler that packs many
// short pairs per CTA and splits long pairs across a CTA by anti-diagonal wavefront").
//   packed classes (W = 1): every warp owns one scratch slot and pulls pairs of its class largest-first;
//   split classes  (W > 1): every CTA owns one scratch slot, its W warps share each pair it pulls.
#pragma once
#include <atomic>

#include "qp_pair.cuh"

namespace qp {

template <typename R, int C, int W> struct KernelSmem {
    using V2 = typename Traits<R>::vec2;
    static constexpr int kWarps = W == 1 ? kWarpsPerCta : W;
    static constexpr size_t tab = sizeof(V2) * kTabDim * kTabDim;
    static constexpr size_t mbars = 256;   // kWarps * kStages mbarriers
    static constexpr size_t rings = (size_t)kWarps * RingBytes<R, C>::v + RingBytes<R, C>::stage;   // + one zeroed stage
    static_assert(kWarps * kStages * 8 <= (int)mbars, "mbarrier area");
    static constexpr size_t hist = (size_t)kWarps * kTauBins * 4;   // per-warp threshold histogram (memory-limited mode)
    template <int GP> static constexpr size_t coop() { return W > 1 ? ((sizeof(CoopShared<R, GP, W>) + 127) & ~(size_t)127) : 0; }
    template <int GP> static constexpr size_t total() { return tab + mbars + rings + coop<GP>() + hist; }
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
    constexpr size_t kCoop = W > 1 ? ((sizeof(CoopShared<R, GP, W>) + 127) & ~(size_t)127) : 0;
    uint32_t* hist_s = (uint32_t*)(rings + SM::rings + kCoop) + (threadIdx.x >> 5) * kTauBins;
    if (ka.tau_hist != nullptr)
        for (int q = threadIdx.x & 31; q < kTauBins; q += 32) hist_s[q] = 0u;
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
    constexpr int cls = class_index(C, W, sizeof(R) == 8, (MODE & kModeMB) != 0);
    const int unit = W == 1 ? blockIdx.x * kWarpsPerCta + warp : blockIdx.x;   // who owns a scratch slot
    SchedHeader* hdr = ka.hdr;
    if constexpr ((MODE & 3) == kModeDist) {
        // consumer of the fp64 re-evaluation queue (split classes only). Drainers (launched after the fp32 classes have
        // joined: every entry is visible) take list positions with an atomicAdd on the class cursor. Pollers run beside
        // the fp32 kernels that fill the list and must never be what keeps those kernels off the SMs, so a poller
        //   - claims a position only once its entry is visible (compare-and-swap on the cursor): it can leave at any
        //     time without owing the list anything, the drainers take whatever is left;
        //   - leaves when every fp32 class warp has exited and the list is drained, OR after kPollIdleMax polls in a
        //     row that found nothing (~20 ms). The second rule makes the call's progress independent of which CTAs
        //     the hardware makes resident first: however many calls, streams or processes share the device, and
        //     however few SMs the context has, waiting CTAs go away by themselves.
        static_assert(W > 1, "the distance-only kernels are split-class kernels");
        RefineQ& q = hdr->rq;
        const bool poll = ka.refine_pass == 1;
        if (unit >= (poll ? q.Wpoll[cls] : q.W[cls])) return;
        char* slot = ka.slots + (poll ? q.poll_slot0[cls] + (unsigned long long)unit * q.poll_slot_bytes[cls]
                                      : q.slot0[cls] + (unsigned long long)unit * q.slot_bytes[cls]);
        const int32_t* list = refine_list_of(ka, cls);
        for (;;) {
            if (threadIdx.x == 0) {
                int v = -1;
                if (!poll) {
                    v = ld_acquire_gpu(list + atomicAdd(&q.cursor[cls], 1));
                } else {
                    for (int idle = 0;;) {
                        const int pos = ld_acquire_gpu(&q.cursor[cls]);
                        v = ld_acquire_gpu(list + pos);
                        if (v >= 0) {
                            if (atomicCAS(&q.cursor[cls], pos, pos + 1) == pos) break;   // ours
                            idle = 0;                                                    // another consumer took it
                            continue;
                        }
                        if (ld_acquire_gpu(&hdr->producers_done) >= ka.producers_total) {   // nothing more will be queued
                            if (ld_acquire_gpu(list + ld_acquire_gpu(&q.cursor[cls])) >= 0) continue;   // a late entry
                            v = -1;
                            break;
                        }
                        if (++idle > kPollIdleMax) {   // give the SM back; the drainers finish the list
                            v = -1;
                            break;
                        }
                        __nanosleep(2000);
                    }
                }
                cs->next = v;
            }
            cta_sync();
            const int p = cs->next;
            if (p < 0) return;
            process_pair<R, GP, C, MODE, W>(ka, smem_u32(tab), p, slot, lane, warp, ring, cs, hist_s);
            cta_sync();   // every warp is done with the slot and with CoopShared
        }
    } else {
        struct Leave {   // every fp32 class warp reports its exit, whatever path it leaves by (pollers wait for the total)
            SchedHeader* h;
            bool on;
            __device__ ~Leave() {
                if (on && (threadIdx.x & 31) == 0) {   // per warp: the warps of a packed-class CTA leave one by one
                    __threadfence();
                    atomicAdd(&h->producers_done, 1);
                }
            }
        } leave{hdr, ka.producers_total > 0};
        const int granted = hdr->cls_W[cls], count = hdr->cls_count[cls];
        const int32_t* list = ka.order + hdr->cls_start[cls];
        if (unit >= granted) return;
        char* slot = ka.slots + ka.slot_off[hdr->cls_slot0[cls] + unit];
        int* cursor = &hdr->cls_cursor[cls];
        int idx = unit;   // the first `granted` pairs of the (largest-first) list go to units 0..granted-1; the rest are pulled
        while (idx < count) {
            process_pair<R, GP, C, MODE, W>(ka, smem_u32(tab), list[idx], slot, lane, warp, ring, cs, hist_s);
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
        if (ka.tau_hist != nullptr) {   // memory-limited mode: this warp's histogram joins the call's
            __syncwarp();
            for (int q = lane; q < kTauBins; q += 32)
                if (hist_s[q]) atomicAdd(&ka.tau_hist[q], (unsigned long long)hist_s[q]);
        }
    }
}

template <typename R, int GP, int C, int MODE, int W> cudaError_t launch_pair(const KArgs<R>& ka, int grid, cudaStream_t st) {
    constexpr size_t smem = KernelSmem<R, C, W>::template total<GP>();
    // the opt-in to more than 48 KB of dynamic shared memory is per device function AND per device: remember it as
    // one bit per device ordinal (per instantiation), set atomically so that host threads may share the library
    static std::atomic<unsigned long long> attr_devs{0};
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    const unsigned long long bit = 1ull << (dev & 63);
    if (dev >= 64 || !(attr_devs.load(std::memory_order_acquire) & bit)) {
        e = cudaFuncSetAttribute(pair_kernel<R, GP, C, MODE, W>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        if (dev < 64) attr_devs.fetch_or(bit, std::memory_order_release);
    }
    pair_kernel<R, GP, C, MODE, W><<<grid, KernelSmem<R, C, W>::kWarps * 32, smem, st>>>(ka);
    return cudaGetLastError();
}

}  // namespace qp
