// qp_pair.cuh -- one warp (packed classes, W = 1) or the W warps of one CTA (split classes, one column block per
// warp, pipelined anti-diagonal wavefront) take one sequence pair through the whole hot path:
//   forward (pair-HMM + partition function, fused)
//   backward (both models) fused with combine, sparsify, MEA  8(a) a2, a4, a5, a6, a7
//   per-row entry buffers -> CSR (rows, columns ascending)     8(a) a6
// Lane arithmetic lives in qp_lane.h; this file owns the wavefront (who processes which row when), the warp
// shuffles that hand row boundaries to the neighbouring lane, and all global-memory traffic.
//
// MODE selects what a kernel instance writes, at compile time, so that the per-cell code carries no test for an
// output that is not wanted:
//   kModeCsr   CSR + distance                       (production)
//   kModeFull  CSR + distance + optional dense_P and logZ (tests)
//   kModeDist  distance only                        (fp64 re-evaluation of near-identical pairs)
#pragma once
#include <cuda_runtime.h>

#include <type_traits>

#include "qp_internal.h"

namespace qp {

enum : int { kModeCsr = 0, kModeFull = 1, kModeDist = 2 };   // | kModeMB (qp_internal.h): the two-block packed instances

constexpr unsigned kFull = 0xffffffffu;

__device__ __forceinline__ float shfl_up1(float v) { return __shfl_up_sync(kFull, v, 1); }
__device__ __forceinline__ double shfl_up1(double v) { return __shfl_up_sync(kFull, v, 1); }
__device__ __forceinline__ int shfl_up1(int v) { return __shfl_up_sync(kFull, v, 1); }
__device__ __forceinline__ float shfl_dn1(float v) { return __shfl_down_sync(kFull, v, 1); }
__device__ __forceinline__ double shfl_dn1(double v) { return __shfl_down_sync(kFull, v, 1); }
__device__ __forceinline__ int shfl_dn1(int v) { return __shfl_down_sync(kFull, v, 1); }
__device__ __forceinline__ int64_t shfl_dn1(int64_t v) { return (int64_t)__shfl_down_sync(kFull, (long long)v, 1); }

// the values always travel; the exponent only on the steps where the receiver rebuilds its scale factor (the caller
// shuffles it separately, under a warp-uniform test, after ALL unconditional shuffles of the step: one convergence
// check per step instead of one per group)
template <typename R, int G> __device__ __forceinline__ FwdEx<R, G> shfl_up_ex(const FwdEx<R, G>& a) {
    FwdEx<R, G> r;
    r.S = shfl_up1(a.S);
    r.M = shfl_up1(a.M);
#pragma unroll
    for (int g = 0; g < G; ++g) r.Y[g] = shfl_up1(a.Y[g]);
    r.e = 0;
    return r;
}
template <typename R, int G> __device__ __forceinline__ BwdEx<R, G> shfl_dn_ex(const BwdEx<R, G>& a) {
    BwdEx<R, G> r;
    r.TL = shfl_dn1(a.TL);
#pragma unroll
    for (int g = 0; g < G; ++g) r.BY[g] = shfl_dn1(a.BY[g]);
    r.e = 0;
    return r;
}
// "nothing comes in": zero values at the receiving lane's own exponent (so that no rescaling is triggered)
template <typename R, int G> __device__ __forceinline__ void zero_ex(FwdEx<R, G>& a, int e) {
    a.S = a.M = R(0);
#pragma unroll
    for (int g = 0; g < G; ++g) a.Y[g] = R(0);
    a.e = e;
}
template <typename R, int G> __device__ __forceinline__ void zero_ex(BwdEx<R, G>& a, int e) {
    a.TL = R(0);
#pragma unroll
    for (int g = 0; g < G; ++g) a.BY[g] = R(0);
    a.e = e;
}

// boundary column handed from one 32*C-column block to the next (multi-block pairs only), one record per row
template <typename R, int GP> struct FwdBnd {
    FwdEx<R, 2> h;
    FwdEx<R, GP> p;
};
template <typename R, int GP> struct BwdBnd {
    BwdEx<R, 2> h;
    BwdEx<R, GP> p;
    typename Traits<R>::acc_t A;
};

__device__ __forceinline__ int warp_sum(int v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(kFull, v, o);
    return v;
}
__device__ __forceinline__ int warp_excl_scan(int v, int lane) {
    int s = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        int t = __shfl_up_sync(kFull, s, o);
        if (lane >= o) s += t;
    }
    return s - v;
}

template <typename R> __device__ __forceinline__ double log2_real(R v) { return log2((double)v); }

// boundary records are written by lane 31/0 and read by lane 0/31 of the same warp in the next block pass:
// read them word-wise through volatile so a stale L1 line from an earlier pair in the same slot cannot be used
template <typename T> __device__ __forceinline__ T ld_volatile(const T* p) {
    static_assert(sizeof(T) % 4 == 0, "record must be a multiple of 4 bytes");
    T r;
    const volatile uint32_t* s = (const volatile uint32_t*)p;
    uint32_t* d = (uint32_t*)&r;
#pragma unroll
    for (int w = 0; w < (int)(sizeof(T) / 4); ++w) d[w] = s[w];
    return r;
}

// ---- scratch addressing of one (step, lane): see qp_internal.h for the layout ------------------------------
// `lp` points at the lane's first F word of the step: step base + lane * kLaneBytes.
template <typename R> struct Slot;
template <> struct Slot<float> {
    static constexpr int kLaneBytes = 16;                                         // one float4 = two cells
};
template <> struct Slot<double> {
    static constexpr int kLaneBytes = 16;                                         // one double2 = one cell
};
// byte distance from `lp` to the lane's int2 exponent record of the same step
template <typename R, int C> __device__ __forceinline__ int exps_delta(int lane) {
    return (int)exps_offset(C, (int)sizeof(R)) + lane * 8 - lane * Slot<R>::kLaneBytes;
}

// ---- backward F staging: TMA bulk copies (cp.async.bulk) of the step records into a per-warp shared-memory ring ----
// The F words of a step record are contiguous ([units][32 lanes] x 16 bytes), so one bulk copy per unit row brings
// the active lanes' words of step t-kStages+1.. into shared memory while step t is computed; completion is
// signalled on a per-stage mbarrier (complete_tx::bytes). The lanes then read their words with 16-byte LDS.
constexpr int kStages = 4;
template <typename R, int C> struct FUnits {   // 16-byte words per lane and step
    static constexpr int k = f_units(C, (int)sizeof(R));
};
template <typename R, int C> struct RingBytes {
    static constexpr int stage = FUnits<R, C>::k * 512;
    static constexpr int v = kStages * stage;
};

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint32_t mbar, int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(mbar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t mbar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(mbar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t mbar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst),
                 "l"(src), "r"(bytes), "r"(mbar)
                 : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t mbar, uint32_t parity) {
    asm volatile(
        "{\n\t.reg .pred P1;\n\tLAB_WAIT:\n\tmbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n\t@P1 bra DONE;\n\t"
        "bra LAB_WAIT;\n\tDONE:\n\t}" ::"r"(mbar),
        "r"(parity)
        : "memory");
}
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async;" ::: "memory"); }

// per-warp ring state; the sequence numbers run over the warp's whole lifetime (stage = seq % kStages,
// parity = (seq / kStages) & 1), copies are consumed in the order they were issued
struct FRing {
    uint32_t data;     // shared-memory address of the ring
    uint32_t mbar;     // shared-memory address of kStages mbarriers
    uint32_t zeros;    // shared-memory address of a zeroed region as large as one stage (shared by the CTA)
    uint32_t issued, waited;
};

// one unit (16 bytes) of a lane's F words, as (F_hmm, F_pf) per cell
template <typename R> struct FWord;
template <> struct FWord<float> {
    float4 v;
    __device__ __forceinline__ Traits<float>::vec2 pair(int k) const {   // (F_hmm, F_pf) of column k: a register pair
        Traits<float>::vec2 r;
        r.x = (k & 1) ? v.z : v.x;
        r.y = (k & 1) ? v.w : v.y;
        return r;
    }
    static __device__ __forceinline__ int unit_of(int k) { return k >> 1; }
    // columns are walked downwards: a unit starts at its odd column, or at the last column of an odd-width stripe
    static __device__ __forceinline__ bool first_of_unit(int k, int C) { return (k & 1) == 1 || k == C - 1; }
};
template <> struct FWord<double> {
    double2 v;
    __device__ __forceinline__ Traits<double>::vec2 pair(int) const {
        Traits<double>::vec2 r;
        r.x = v.x;
        r.y = v.y;
        return r;
    }
    static __device__ __forceinline__ int unit_of(int k) { return k; }
    static __device__ __forceinline__ bool first_of_unit(int, int) { return true; }
};
// one (em_hmm, em_pf) entry of the emission table; explicit shared-space loads keep the generic->shared address
// conversion out of the step loop
__device__ __forceinline__ Traits<float>::vec2 lds_em(uint32_t addr, float) {
    Traits<float>::vec2 v;
    asm volatile("ld.shared.v2.f32 {%0,%1}, [%2];" : "=f"(v.x), "=f"(v.y) : "r"(addr));
    return v;
}
__device__ __forceinline__ Traits<double>::vec2 lds_em(uint32_t addr, double) {
    Traits<double>::vec2 v;
    asm volatile("ld.shared.v2.f64 {%0,%1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(addr));
    return v;
}
__device__ __forceinline__ void lds16(float4& v, uint32_t addr) {
    asm volatile("ld.shared.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(addr));
}
__device__ __forceinline__ void lds16(double2& v, uint32_t addr) {
    asm volatile("ld.shared.v2.f64 {%0,%1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(addr));
}

// append a kept posterior to its row's entry buffer and advance the buffer pointer: predicated 8-byte store and
// predicated 64-bit add, no branch. (A 32-bit entry count + mad.wide address under the predicate is three instructions
// instead of seven in SASS, but needs one more live register and the C = 8..12 kernels then spill: measured +20 %.)
__device__ __forceinline__ void st_entry_adv(char*& ptr, float val, int col, bool keep) {
    asm volatile(
        "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %3, 0;\n\t@p st.global.v2.b32 [%0], {%1, %2};\n\t@p add.s64 %0, %0, 8;\n\t}"
        : "+l"(ptr)
        : "r"(__float_as_int(val)), "r"(col), "r"((int)keep)
        : "memory");
}
// entry buffers and row counts are written by one lane and read by another lane of the same warp: read them from L2
__device__ __forceinline__ float4 ld_cg_f4(const void* p) { return __ldcg((const float4*)p); }

// ---- split pairs: W warps of one CTA share a pair (north_star: "splits long pairs across a CTA by anti-diagonal
// wavefront"). Warp w takes column block b0+w of the current group of W blocks; the block boundary (the values lane 31
// hands to lane 0 of the next block forward, lane 0 to lane 31 of the previous block backward) travels through a
// shared-memory ring of kDepth rows per neighbour pair, guarded by two counters: rows produced (release/acquire)
// and rows consumed (back-pressure). Every warp runs free; in steady state block w+1 trails block w by 33 steps, so
// one pass over a group takes rows + 32*(active warps) steps instead of (rows + 32) * blocks.
template <typename R, int GP, int W> struct CoopShared {
    static constexpr int kDepth = 32;
    union Rec {
        FwdBnd<R, GP> f;
        BwdBnd<R, GP> b;
    };
    Rec ring[W > 1 ? W - 1 : 1][kDepth];   // channel c: between warp c and warp c+1
    int prod[W], cons[W];
    R z[2];                                // forward totals (mantissas) and their exponents, from the last block's warp
    int ez[2];
    unsigned long long poff;               // CSR staging-pool offset of the pair
    int ok;
    int next;                              // next pair index (CTA-wide pull)
};
__device__ __forceinline__ int ld_acquire_cta(const int* p) {
    int v;
    asm volatile("ld.acquire.cta.shared.s32 %0, [%1];" : "=r"(v) : "r"(smem_u32(p)) : "memory");
    return v;
}
__device__ __forceinline__ void st_release_cta(int* p, int v) {
    asm volatile("st.release.cta.shared.s32 [%0], %1;" ::"r"(smem_u32(p)), "r"(v) : "memory");
}
__device__ __forceinline__ void cta_sync() { __syncthreads(); }

// Residue codes of the rows: lane l works on row t-l, so a lane's next row is its neighbour's current one. The code
// travels with the wavefront by shuffle; only the entering lane (lane 0 forward, lane 31 backward) takes a new
// code, from a 32-row chunk that the warp loads (coalesced) one chunk ahead of its use.

// re-evaluation list of split fp64 class cls (kNumPacked..kNumClasses-1)
template <typename R> __host__ __device__ __forceinline__ int32_t* refine_list_of(const KArgs<R>& ka, int cls) {
    return ka.refine_list + (int64_t)(cls - kNumPacked) * ka.refine_stride;
}
__device__ __forceinline__ void st_release_gpu(int32_t* p, int32_t v) {
    asm volatile("st.release.gpu.global.s32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
__device__ __forceinline__ int32_t ld_acquire_gpu(const int32_t* p) {
    int32_t v;
    asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}

// ---------------------------------------------------------------------------------------------------------
// the pair pipeline
// ---------------------------------------------------------------------------------------------------------
template <typename R, int GP, int C, int MODEX, int W>
__device__ void process_pair(const KArgs<R>& ka, const uint32_t tab /*shared address of the emission table*/, int p,
                             char* slot, int lane, int warp, FRing& ring, CoopShared<R, GP, W>* cs,
                             uint32_t* hist_s /*this warp's threshold histogram in shared memory*/) {
    using V2 = typename Traits<R>::vec2;
    using Acc = typename Traits<R>::acc_t;
    using SL = Slot<R>;
    constexpr int MODE = MODEX & 3;                  // what is written
    constexpr bool kMB = (MODEX & kModeMB) != 0;     // packed class whose pairs have two column blocks
    constexpr int RB = (int)sizeof(R);
    constexpr int GH = 2;
    constexpr bool kCsr = MODE != kModeDist;
    constexpr int kDepth = CoopShared<R, GP, W>::kDepth;
    constexpr bool kSplit = W > 1;
    if constexpr (!kSplit) warp = 0;

    const PairInfo pi = ka.info[p];
    const int n = pi.n, m = pi.m;
    // column blocks (column 0 included); a one-block packed class only takes pairs that fit one block (choose_class)
    const int nb = (kSplit || kMB) ? (m + 1 + 32 * C - 1) / (32 * C) : 1;
    constexpr int kEm = (int)sizeof(V2);
    const uint8_t* __restrict__ xs = ka.seqs + pi.xoff;
    const uint8_t* __restrict__ ys = ka.seqs + pi.yoff;
    constexpr int stride = (int)step_stride(C, RB);
    const int64_t blk_bytes = (int64_t)num_steps(n) * stride;
    const int cols_last = (m + 1) - (nb - 1) * 32 * C;   // columns (incl. column 0) that fall in the last block
    const int lz = (cols_last - 1) / C, kz = (cols_last - 1) % C;   // lane / stripe offset of column m
    const int mask = ka.rescale_mask;
    const int dE = exps_delta<R, C>(lane);
    char* bnd0 = slot + (int64_t)nb * blk_bytes;
    char* bnd1 = bnd0 + (int64_t)(n + 1) * bnd_rec_bytes(RB);
    int range_flag = 0;
    // residue bytes index the 32 x 32 emission table in shared memory: clamp them so that an invalid code (>= 32; the
    // call then ends with QP_ERR_BAD_RESIDUE, k_check_residues) can never address outside the table
    auto xcode_at = [&](int i) -> int { return (i >= 1 && i <= n) ? min((int)__ldg(xs + i - 1), kSentinel) : kSentinel; };

    // =========================================== forward ===================================================
    R zcap_h = R(0), zcap_p = R(0);
    int ez_h = 0, ez_p = 0;
    for (int b0 = 0; b0 < nb; b0 += W) {
      if constexpr (kSplit) {   // fresh ring counters for this group of W blocks
        cta_sync();
        if (lane == 0) cs->prod[warp] = cs->cons[warp] = 0;
        cta_sync();
      }
      const int b = b0 + warp;
      if (b < nb) {
        FwdBoth<R, GP, C> FB;   // both automata of this lane (qp_both.cuh)
        FB.init();
        int ycode[C];   // byte offset of the column's residue inside a table row
#pragma unroll
        for (int k = 0; k < C; ++k) {
            int j = b * 32 * C + lane * C + k;
            ycode[k] = ((j >= 1 && j <= m) ? min((int)ys[j - 1], kSentinel) : kSentinel) * kEm;
        }
        const bool last = (b == nb - 1);
        const int tend = n + (last ? lz : 31);
        bool rare_h = false, rare_p = false;   // warp-uniform: some lane needs the second scale factor
        // boundary columns between groups of W blocks go through the slot (ping-pong by group); inside a group
        // (split pairs) through the shared-memory rings
        const int grp = b0 / W;
        const FwdBnd<R, GP>* bin = (const FwdBnd<R, GP>*)((grp & 1) ? bnd0 : bnd1);   // written by the previous group
        FwdBnd<R, GP>* bout = (FwdBnd<R, GP>*)((grp & 1) ? bnd1 : bnd0);
        const bool in_ring = kSplit && warp > 0, out_ring = kSplit && warp < W - 1;
        char* lp = slot + (int64_t)b * blk_bytes + lane * SL::kLaneBytes;   // this lane's F words of step t
        const bool colact = b * 32 * C + lane * C <= m;   // lanes that hold only padding columns store nothing
        // row codes: every lane starts on a row <= 0; lane 0 enters row t+1 at the end of step t
        int xcode = kSentinel;
        int chunk = xcode_at(lane + 1), chunk_next = xcode_at(lane + 33);
        for (int t = 0; t <= tend; ++t, lp += stride) {
            const int i = t - lane;
            const bool active = (unsigned)i <= (unsigned)n;
            // warp-uniform (FwdModel::prepare): lanes enter their first row while t < 32; scales change on the
            // renormalisation step and the step after it; lane 0 of a later block of a multi-block pair loses its input
            // once it is past row n
            const bool recompute = (t & mask) <= 1 || ((kSplit || kMB) && b > 0 && t > n);
            const bool prep = recompute || t < 32;
            FwdEx<R, GH> rh = shfl_up_ex(FB.exh());
            FwdEx<R, GP> rp = shfl_up_ex(FB.exp());
            const uint32_t row = tab + xcode * (kTabDim * kEm);
            {
                const int feed = __shfl_sync(kFull, chunk, t & 31);
                const int up = __shfl_up_sync(kFull, xcode, 1);
                if (prep) {
                    rh.e = shfl_up1(FB.exh().e);
                    rp.e = shfl_up1(FB.exp().e);
                }
                xcode = lane == 0 ? feed : up;
                if ((t & 31) == 31) {   // warp-uniform
                    chunk = chunk_next;
                    chunk_next = xcode_at(t + 34 + lane);
                }
            }
            bool zero_in = lane == 0;   // nothing comes in from the left of the first block
            if (b > 0) {                // warp-uniform: lane 0 takes the boundary column of the previous block
                zero_in = lane == 0 && !active;
                if (in_ring) {
                    if (t <= n) {       // warp-uniform: lane 0 is on row t; wait until the left block has produced it
                        while (ld_acquire_cta(&cs->prod[warp - 1]) <= t) {}
                        if (lane == 0) {
                            const FwdBnd<R, GP> rec = cs->ring[warp - 1][t % kDepth].f;
                            rh = rec.h;
                            rp = rec.p;
                            st_release_cta(&cs->cons[warp - 1], t + 1);
                        }
                    }
                } else if (lane == 0 && active) {
                    const FwdBnd<R, GP> rec = ld_volatile(bin + i);
                    rh = rec.h;
                    rp = rec.p;
                }
            }
            if (prep) {
                const bool resc = (t & mask) == 0;
                FB.prepare(rh, rp, i == 0, resc, recompute, zero_in, range_flag);
                rare_h = __any_sync(kFull, FB.rare_h());
                rare_p = __any_sync(kFull, FB.rare_p());
            }
            FB.load(rh, rp, rare_h, rare_p, ka.wh, ka.wp, ka.w2);
            const bool special = (b == 0 && t == 0) || (last && t == tend);   // warp-uniform
            FwdSpecial sp;
            sp.start = sp.capture = false;
            sp.kz = kz;
            if (special) {
                sp.start = b == 0 && lane == 0 && i == 0;
                sp.capture = last && lane == lz && i == n;
            }
            const bool st_on = active && colact;
            auto body = [&](auto SPEC) {
                constexpr bool S = decltype(SPEC)::value;
                R dh = R(0), dp = R(0);
                [[maybe_unused]] V2 prev;
#pragma unroll
                for (int k = 0; k < C; ++k) {
                    const V2 em = lds_em(row + ycode[k], R(0));
                    const V2 o = FB.template cell<S>(k, em, ka.wh, ka.wp, ka.w2, sp, S ? zcap_h : dh, S ? zcap_p : dp);
                    if constexpr (sizeof(R) == 4) {
                        if (k & 1) {
                            if (st_on) __stcs((float4*)(lp + (k >> 1) * 512), make_float4(prev.x, prev.y, o.x, o.y));
                        } else if (k == C - 1) {   // odd stripe width: the last word is half used
                            if (st_on) __stcs((float4*)(lp + (k >> 1) * 512), make_float4(o.x, o.y, 0.f, 0.f));
                        } else {
                            prev = o;
                        }
                    } else {
                        if (st_on) *(V2*)(lp + k * 512) = o;
                    }
                }
            };
            if (special) body(std::true_type{});
            else body(std::false_type{});
            FB.end();
            // exponents: constant over a renormalisation period, recorded on its last step (all lanes: a lane whose
            // last row fell inside the period has kept its exponent since)
            if ((t & mask) == mask || t == tend) *(int2*)(lp + dE) = make_int2(FB.eh(), FB.ep());
            if (nb > 1 && !last) {
                if (out_ring) {
                    const int i31 = t - 31;   // warp-uniform: the row lane 31 has just finished
                    if (i31 >= 0 && i31 <= n) {
                        if (i31 >= kDepth)    // back-pressure: the ring entry must have been consumed
                            while (ld_acquire_cta(&cs->cons[warp]) < i31 - kDepth + 1) {}
                        if (lane == 31) {
                            FwdBnd<R, GP>& rec = cs->ring[warp][i31 % kDepth].f;
                            rec.h = FB.exh();
                            rec.p = FB.exp();
                            st_release_cta(&cs->prod[warp], i31 + 1);
                        }
                    }
                } else if (lane == 31 && active) {
                    bout[i].h = FB.exh();
                    bout[i].p = FB.exp();
                }
            }
        }
        if (last) {
            ez_h = FB.eh();
            ez_p = FB.ep();
            if constexpr (kSplit) {   // the forward totals live in lane lz of this warp: publish them to the CTA
                if (lane == lz) {
                    cs->z[0] = zcap_h;
                    cs->z[1] = zcap_p;
                    cs->ez[0] = ez_h;
                    cs->ez[1] = ez_p;
                }
            }
        }
        if (nb > 1) __syncwarp();   // lane 31's boundary column must be visible to lane 0 of the next block
      }
    }
    // Z = Zm * 2^eZ with Zm in [1,2); every lane gets a copy
    if constexpr (kSplit) {
        cta_sync();   // also orders the boundary column of the last group's writes before the backward reads
        zcap_h = cs->z[0];
        zcap_p = cs->z[1];
        ez_h = cs->ez[0];
        ez_p = cs->ez[1];
    } else {
        zcap_h = __shfl_sync(kFull, zcap_h, lz);
        zcap_p = __shfl_sync(kFull, zcap_p, lz);
        ez_h = __shfl_sync(kFull, ez_h, lz);
        ez_p = __shfl_sync(kFull, ez_p, lz);
    }
    {
        int kh = expo(zcap_h), kp = expo(zcap_p);
        if (kh == kZeroExp || kp == kZeroExp) {   // total underflow: weights outside the supported range
            range_flag = 1;
            kh = kp = 0;
            zcap_h = zcap_p = R(1);
        }
        zcap_h *= pow2i(-kh, R(0));
        zcap_p *= pow2i(-kp, R(0));
        ez_h += kh;
        ez_p += kp;
    }
    const R invZh = inv_z_rms(zcap_h), invZp = inv_z_rms(zcap_p);

    // ================================ backward + combine + sparsify + MEA ================================
    const int minnm = n < m ? n : m;
    int sbits = (int)(8 * sizeof(Acc)) - 2;   // fixed-point fraction bits of the MEA accumulator
    {
        int need = 1;
        while ((1 << need) <= minnm) ++need;   // bits for the integer part
        sbits -= need;
        const int cap = sizeof(R) == 4 ? 20 : 40;   // fp32: P*2^s must stay below 2^22 for the magic rounding
        if (sbits > cap) sbits = cap;
    }
    const R mea_scale = (R)ldexp(1.0, sbits);
    float* dense = nullptr;
    if constexpr (MODE == kModeFull) dense = ka.dense_P != nullptr ? ka.dense_P + ka.dense_off[p] : nullptr;
    R zb_h = R(0), zb_p = R(0);
    int ezb_h = 0, ezb_p = 0;
    int nnz_lane = 0;
    Acc mea = 0;
    for (int b0 = ((nb - 1) / W) * W; b0 >= 0; b0 -= W) {
      if constexpr (kSplit) {   // fresh ring counters for this group of W blocks
        cta_sync();
        if (lane == 0) cs->prod[warp] = cs->cons[warp] = 0;
        cta_sync();
      }
      const int b = b0 + warp;
      if (b < nb) {
        BwdBoth<R, GP, C> BB;   // both automata of this lane (qp_both.cuh)
        BB.init();
        Acc An[C];
        int ycode[C];
#pragma unroll
        for (int k = 0; k < C; ++k) {
            An[k] = 0;
            int j = b * 32 * C + lane * C + k;
            ycode[k] = ((j >= 1 && j <= m) ? min((int)ys[j - 1], kSentinel) : kSentinel) * kEm;
        }
        Acc Adin = 0, exA = 0;
        bool rare_h = false, rare_p = false;   // warp-uniform, see the forward loop
        PScale<R> psh, psp;                    // posterior scale of this lane: changes only when an exponent does
        psh.c = psp.c = R(0);
        const bool last = (b == nb - 1);
        const int tstart = n + (last ? lz : 31);
        const int grp = b0 / W;
        const BwdBnd<R, GP>* bin = (const BwdBnd<R, GP>*)((grp & 1) ? bnd0 : bnd1);   // written by the next group
        BwdBnd<R, GP>* bout = (BwdBnd<R, GP>*)((grp & 1) ? bnd1 : bnd0);
        const bool in_ring = kSplit && warp < W - 1, out_ring = kSplit && warp > 0;
        const int jbase = b * 32 * C + lane * C;
        const bool colact = jbase <= m;   // lanes that hold only padding columns: nothing was stored for them
        // row codes: lane l starts on row tstart-l; lane 31 enters row t-32 at the end of step t
        int xcode = xcode_at(tstart - lane);
        int chunk = xcode_at(tstart - 32 - lane), chunk_next = xcode_at(tstart - 64 - lane);
        // F words: one bulk copy per step brings the whole F area of a step record into the ring, kStages-1 steps
        // ahead of the wavefront (see FRing). Lanes whose row is outside 0..n at that step, and lanes that hold only
        // padding columns, never wrote their words: they read zeros from a shared zero region instead (posterior 0).
        // Exponent records exist on the last step of every renormalisation period (and of the block); they are
        // fetched one step ahead.
        char* lp = slot + (int64_t)b * blk_bytes + (int64_t)tstart * stride + lane * SL::kLaneBytes;
        constexpr int kUnits = FUnits<R, C>::k;
        const char* blk0 = slot + (int64_t)b * blk_bytes;
        auto issue = [&](int tt) {   // bulk-copy the F area of step tt
            const uint32_t st = ring.issued % kStages;
            if (lane == 0) {   // one lane issues: the copy instruction takes uniform operands
                // (copying only the on-grid lanes' share of every unit row on the ramp steps -- kUnits small copies
                // instead of one -- saves ~4 % of the reads and was measured no faster: round 2)
                const uint32_t mb = ring.mbar + st * 8;
                mbar_expect_tx(mb, kUnits * 512);
                bulk_g2s(ring.data + st * (kUnits * 512), blk0 + (int64_t)tt * stride, kUnits * 512, mb);
            }
            ++ring.issued;
        };
        fence_proxy_async();   // the forward pass wrote the records through the generic proxy
        __syncwarp();
#pragma unroll 1
        for (int d = 0; d < kStages; ++d)
            if (tstart - d >= 0) issue(tstart - d);
        int2 eF = *(const int2*)(lp + dE), eFn = eF;
        // entries of row i = t - lane go to step record i + 32 of this block (qp_internal.h); the row's running
        // entry count travels down the lanes with the row
        const int64_t dRow = (int64_t)(32 - lane) * stride - lane * SL::kLaneBytes;
        int ecnt = 0;
        int32_t* rowcnt = (int32_t*)(slot + rowcnt_offset(n, C, nb, RB)) + (int64_t)b * (n + 1);
        for (int t = tstart; t >= 0; --t, lp -= stride) {
            const int i = t - lane;
            const bool active = (unsigned)i <= (unsigned)n;
            const bool more = t > 0;
            const bool enext = more && (((t - 1) & mask) == mask);   // warp-uniform: step t-1 holds a record
            if (enext) eFn = *(const int2*)(lp - stride + dE);
            // warp-uniform (FwdModel::prepare): lanes enter their first row (row n) while t >= n; scales change on the
            // renormalisation step and the step after it (that is also where the recorded forward exponents change);
            // lane 31 of an earlier block of a multi-block pair loses its input once it is past row 0
            const bool recompute = (t & mask) >= mask - 1 || ((kSplit || kMB) && !last && t < 32);
            const bool prep = recompute || t >= n;
            BwdEx<R, GH> rh = shfl_dn_ex(BB.exh());
            BwdEx<R, GP> rp = shfl_dn_ex(BB.exp());
            Acc rA = shfl_dn1(exA);
            if constexpr (kCsr) ecnt = shfl_dn1(ecnt);
            const uint32_t row = tab + xcode * (kTabDim * kEm);
            {
                const int sdn = tstart - t;
                const int feed = __shfl_sync(kFull, chunk, sdn & 31);
                const int dn = __shfl_down_sync(kFull, xcode, 1);
                if (prep) {
                    rh.e = shfl_dn1(BB.exh().e);
                    rp.e = shfl_dn1(BB.exp().e);
                }
                if (lane == 31) rA = 0;
                if constexpr (kCsr) {
                    if (lane == 31) ecnt = 0;
                }
                xcode = lane == 31 ? feed : dn;
                if ((sdn & 31) == 31) {   // warp-uniform
                    chunk = chunk_next;
                    chunk_next = xcode_at(t - 65 - lane);
                }
            }
            bool zero_in = lane == 31;   // nothing comes in from the right of the last block
            if (!last) {                 // warp-uniform: lane 31 takes the boundary column of the next block
                zero_in = lane == 31 && !active;
                if (in_ring) {
                    const int i31 = t - 31;   // warp-uniform: the row lane 31 is on; rows arrive in the order n, n-1, ...
                    if (i31 >= 0 && i31 <= n) {
                        const int seq = n - i31;
                        while (ld_acquire_cta(&cs->prod[warp]) <= seq) {}
                        if (lane == 31) {
                            const BwdBnd<R, GP> rec = cs->ring[warp][seq % kDepth].b;
                            rh = rec.h;
                            rp = rec.p;
                            rA = rec.A;
                            st_release_cta(&cs->cons[warp], seq + 1);
                        }
                    }
                } else if (lane == 31 && active) {
                    const BwdBnd<R, GP> rec = ld_volatile(bin + i);
                    rh = rec.h;
                    rp = rec.p;
                    rA = rec.A;
                }
            }
            if (prep) {
                const bool resc = (t & mask) == mask;
                BB.prepare(rh, rp, i == n, resc, recompute, zero_in, range_flag);
                rare_h = __any_sync(kFull, BB.rare_h());
                rare_p = __any_sync(kFull, BB.rare_p());
                const bool bad_h = psh.set(eF.x + BB.eh() - ez_h, invZh);
                const bool bad_p = psp.set(eF.y + BB.ep() - ez_p, invZp);
                if ((bad_h || bad_p) && active && colact) range_flag = 1;   // padding lanes hold B = 0 at exponent 0
            }
            BB.load(rh, rp, rare_h, rare_p);
            // this step's F words have landed?
            const uint32_t stg = ring.waited % kStages;
            mbar_wait(ring.mbar + stg * 8, (ring.waited / kStages) & 1);
            ++ring.waited;
            const uint32_t sF = ((active && colact) ? ring.data + stg * (kUnits * 512) : ring.zeros) + lane * 16;
            const bool special = (last && t == tstart) || (b == 0 && t == 0);   // warp-uniform
            BwdSpecial sp;
            sp.end = sp.capture = false;
            sp.kz = kz;
            if (special) {
                sp.end = last && lane == lz && i == n;
                sp.capture = b == 0 && lane == 0 && i == 0;
            }
            Acc Adiag = Adin, Aright = rA;
            const bool row_ok = (i >= 1) && (i <= n);
            char* ep = lp + dRow + (int64_t)ecnt * 8;   // next free entry of this lane's row
            auto body = [&](auto SPEC) {
                constexpr bool S = decltype(SPEC)::value;
                FWord<R> Fw, Fn;   // the unit in use and the next one, read one unit ahead
                lds16(Fn.v, sF + (kUnits - 1) * 512);
#pragma unroll
                for (int k = C - 1; k >= 0; --k) {
                    if (FWord<R>::first_of_unit(k, C)) {
                        Fw = Fn;
                        if (FWord<R>::unit_of(k) > 0) lds16(Fn.v, sF + (FWord<R>::unit_of(k) - 1) * 512);
                    }
                    // the two backward recurrences
                    const V2 em = lds_em(row + ycode[k], R(0));
                    R zh = R(0), zp = R(0);
                    const V2 bm = BB.template cell<S>(k, em, ka.wh, ka.wp, ka.w2, sp, zh, zp);
                    if (S && sp.capture && k == 0) {
                        zb_h = zh;
                        zb_p = zp;
                        ezb_h = BB.eh();
                        ezb_p = BB.ep();
                    }
                    // combine, expected-accuracy max-plus, threshold + append to the row's entry buffer
                    const V2 pm = BB.posterior(Fw.pair(k), bm, psh, psp);
                    const R P = combine_rms(pm.x, pm.y);
                    const Acc q = quantise(P, mea_scale);
                    Acc a = Adiag + q;
                    a = a > An[k] ? a : An[k];
                    a = a > Aright ? a : Aright;
                    Adiag = An[k];
                    An[k] = a;
                    Aright = a;
                    if constexpr (kCsr) {
                        const bool keep = P >= ka.tau;
                        st_entry_adv(ep, (float)P, jbase + k - 1, keep);   // 0-based column in y
                    }
                    if constexpr (MODE == kModeFull) {
                        const int j = jbase + k;
                        if (dense != nullptr && row_ok && j >= 1 && j <= m) dense[(int64_t)(i - 1) * m + (j - 1)] = (float)P;
                    }
                }
            };
            if (special) body(std::true_type{});
            else body(std::false_type{});
            if (enext) eF = eFn;
            __syncwarp();   // every lane has read its words of this stage: refill it
            if (t >= kStages) issue(t - kStages);
            BB.end();
            exA = An[0];
            Adin = rA;
            if constexpr (kCsr) {
                ecnt = (int)((ep - (lp + dRow)) >> 3);
                if (lane == 0 && active) {   // row i of this block is complete
                    rowcnt[i] = ecnt;
                    nnz_lane += ecnt;
                }
            }
            if (nb > 1 && b > 0) {
                if (out_ring) {
                    if (t <= n) {   // warp-uniform: lane 0 has just finished row t
                        const int seq = n - t;
                        if (seq >= kDepth)
                            while (ld_acquire_cta(&cs->cons[warp - 1]) < seq - kDepth + 1) {}
                        if (lane == 0) {
                            BwdBnd<R, GP>& rec = cs->ring[warp - 1][seq % kDepth].b;
                            rec.h = BB.exh();
                            rec.p = BB.exp();
                            rec.A = exA;
                            st_release_cta(&cs->prod[warp - 1], seq + 1);
                        }
                    }
                } else if (lane == 0 && active) {
                    bout[i].h = BB.exh();
                    bout[i].p = BB.exp();
                    bout[i].A = exA;
                }
            }
        }
        if (b == 0) mea = An[0];   // lane 0 holds A'(0,0) = A(n,m)
        if (nb > 1) __syncwarp();
      }
    }
    mea = __shfl_sync(kFull, mea, 0);   // split pairs: only warp 0 (block 0) holds it, and only warp 0 uses it
    const double dist = 1.0 - (double)mea / (ldexp(1.0, sbits) * (double)minnm);

    if (__any_sync(kFull, range_flag)) {
        if (lane == 0 && atomicCAS(&ka.hdr->status[0], 0, -8 /*QP_ERR_RANGE*/) == 0) ka.hdr->status[1] = p;
    }

    // ---- distance d = 1 - A(n,m)/min(n,m), both orientations; near-identical pairs are queued for fp64 --------
    if (lane == 0 && warp == 0) {
        const int xi = ka.pairs[2 * (int64_t)p], yi = ka.pairs[2 * (int64_t)p + 1];
        ka.dist[(int64_t)xi * ka.k + yi] = (float)dist;
        ka.dist[(int64_t)yi * ka.k + xi] = (float)dist;
        // fp32 distance error grows like sqrt(n + m) (measured <= 3.7e-8 * sqrt(n + m) absolute): beyond 4000 rows +
        // columns the re-evaluation limit grows with it, so that relative 1e-5 keeps its margin on very long pairs
        const float lim = ka.refine_below * fmaxf(1.f, sqrtf((float)(n + m) * (1.f / 4000.f)));
        if (MODE != kModeDist && sizeof(R) == 4 && (float)dist < lim) {
            int nbd;
            const int c64 = choose_class(n, m + 1, ka.refine_cmask, true, &nbd);
            RefineQ& q = ka.hdr->rq;
            const int pos = atomicAdd(&q.count[c64], 1);
            atomicMax(&q.slot_bytes[c64], (unsigned long long)slot_bytes(n, class_C(c64, true), nbd, 8));
            // publish: the fp64 kernel that picks the entry up overwrites the distance written above
            st_release_gpu(refine_list_of(ka, c64) + pos, p);
        }
    }

    // ---- logZ (tests): undo the background normalisation, ln Z = ln2*(log2 Zm + eZ) + sum lx ----------------
    if constexpr (MODE == kModeFull) {
        if (ka.logZ != nullptr && warp == 0) {
            double ch = 0.0, cp = 0.0;
            for (int q = lane; q < n; q += 32) { ch += ka.lx_h[xs[q] & 31]; cp += ka.lx_p[xs[q] & 31]; }
            for (int q = lane; q < m; q += 32) { ch += ka.lx_h[ys[q] & 31]; cp += ka.lx_p[ys[q] & 31]; }
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
                ch += __shfl_xor_sync(kFull, ch, o);
                cp += __shfl_xor_sync(kFull, cp, o);
            }
            zb_h = __shfl_sync(kFull, zb_h, 0);
            zb_p = __shfl_sync(kFull, zb_p, 0);
            ezb_h = __shfl_sync(kFull, ezb_h, 0);
            ezb_p = __shfl_sync(kFull, ezb_p, 0);
            if (lane == 0) {
                const double ln2 = 0.69314718055994530942;
                double* o = ka.logZ + 4 * (int64_t)p;
                o[0] = ln2 * (log2_real(zcap_h) + ez_h) + ch;
                o[1] = ln2 * (log2_real(zb_h) + ezb_h) + ch;
                o[2] = ln2 * (log2_real(zcap_p) + ez_p) + cp;
                o[3] = ln2 * (log2_real(zb_p) + ezb_p) + cp;
            }
        }
    }

    // ---- CSR: row counts -> row_ptr, entry buffers -> staging pool, rows ascending, columns ascending -----------
    // 32 rows at a time, one row per lane. A row's entries sit in its buffer(s) highest column first; blocks are
    // walked in ascending order and every buffer backwards, four entries (one 32-byte sector) per load pair.
    if constexpr (kCsr && kSplit) {
        // split pairs: warp 0 turns the row counts into row_ptr and reserves the pool range, then all W warps
        // move the entry buffers, 32 rows per warp at a time
        cta_sync();   // entry buffers and row counts were written by all warps of the CTA
        int32_t* rp = ka.row_ptr + ka.pair_row_base[p];
        const int32_t* rowcnt = (const int32_t*)(slot + rowcnt_offset(n, C, nb, RB));
        if (warp == 0) {
            int running = 0;
            for (int i0 = 1; i0 <= n; i0 += 32) {
                const int i = i0 + lane;
                const bool valid = i <= n;
                int c = 0;
                for (int b = 0; b < nb; ++b) c += valid ? __ldcg(rowcnt + (int64_t)b * (n + 1) + i) : 0;
                const int ex = warp_excl_scan(c, lane);
                if (valid) rp[i - 1] = running + ex;
                running += __shfl_sync(kFull, ex + c, 31);
            }
            if (lane == 0) {
                const unsigned long long poff = atomicAdd(&ka.hdr->pool_cursor, (unsigned long long)running);
                const bool ok = (long long)(poff + (unsigned long long)running) <= (long long)ka.pool_cap;
                if (!ok && atomicCAS(&ka.hdr->status[0], 0, -6 /*QP_ERR_NNZ_CAPACITY*/) == 0) ka.hdr->status[1] = p;
                cs->poff = poff;
                cs->ok = ok;
                rp[n] = running;
                ka.nnz[p] = running;
                ka.pool_off[p] = (int64_t)poff;
            }
        }
        cta_sync();
        if (cs->ok) {
            float2* pool = ka.pool + cs->poff;   // (value, column bits) per entry
            for (int i0 = 1 + 32 * warp; i0 <= n; i0 += 32 * W) {
                const int i = i0 + lane;
                if (i > n) continue;
                int d = __ldcg(rp + i - 1);
                for (int b = 0; b < nb; ++b) {
                    const int cb = __ldcg(rowcnt + (int64_t)b * (n + 1) + i);
                    const char* buf = slot + (int64_t)b * blk_bytes + (int64_t)(i + 32) * stride;
                    for (int g = (cb - 1) >> 2; g >= 0; --g) {
                        const float4 lo = ld_cg_f4(buf + g * 32), hi = ld_cg_f4(buf + g * 32 + 16);
                        const int q = 4 * g;
                        if (q + 3 < cb) { pool[d] = make_float2(hi.z, hi.w); ++d; }
                        if (q + 2 < cb) { pool[d] = make_float2(hi.x, hi.y); ++d; }
                        if (q + 1 < cb) { pool[d] = make_float2(lo.z, lo.w); ++d; }
                        pool[d] = make_float2(lo.x, lo.y); ++d;
                    }
                }
            }
        }
    } else if constexpr (kCsr) {
        __syncwarp();   // entry buffers and row counts were written by other lanes of this warp
        const int nnz = warp_sum(nnz_lane);
        unsigned long long poff = 0;
        if (lane == 0) poff = atomicAdd(&ka.hdr->pool_cursor, (unsigned long long)nnz);
        poff = __shfl_sync(kFull, poff, 0);
        const bool ok = (long long)(poff + (unsigned long long)nnz) <= (long long)ka.pool_cap;
        if (!ok && lane == 0) {
            if (atomicCAS(&ka.hdr->status[0], 0, -6 /*QP_ERR_NNZ_CAPACITY*/) == 0) ka.hdr->status[1] = p;
        }
        int32_t* rp = ka.row_ptr + ka.pair_row_base[p];
        float2* pool = ka.pool + poff;   // (value, column bits) per entry: one 8-byte store each
        const int32_t* rowcnt = (const int32_t*)(slot + rowcnt_offset(n, C, nb, RB));
        if constexpr (kMB) {
            // two blocks (packed class, wide pair): plain walk, rows 32 at a time, blocks in ascending order
            int running = 0;
            for (int i0 = 1; i0 <= n; i0 += 32) {
                const int i = i0 + lane;
                const bool valid = i <= n;
                int c = 0;
                for (int b = 0; b < nb; ++b) c += valid ? __ldcg(rowcnt + (int64_t)b * (n + 1) + i) : 0;
                const int ex = warp_excl_scan(c, lane);
                int d = running + ex;
                if (valid) rp[i - 1] = d;
                running += __shfl_sync(kFull, ex + c, 31);
                if (ok && valid)
                    for (int b = 0; b < nb; ++b) {
                        const int cb = __ldcg(rowcnt + (int64_t)b * (n + 1) + i);
                        const char* buf = slot + (int64_t)b * blk_bytes + (int64_t)(i + 32) * stride;
                        for (int g = (cb - 1) >> 2; g >= 0; --g) {
                            const float4 lo = ld_cg_f4(buf + g * 32), hi = ld_cg_f4(buf + g * 32 + 16);
                            const int q = 4 * g;
                            if (q + 3 < cb) { pool[d] = make_float2(hi.z, hi.w); ++d; }
                            if (q + 2 < cb) { pool[d] = make_float2(hi.x, hi.y); ++d; }
                            if (q + 1 < cb) { pool[d] = make_float2(lo.z, lo.w); ++d; }
                            pool[d] = make_float2(lo.x, lo.y); ++d;
                        }
                    }
            }
            if (lane == 0) {
                rp[n] = running;
                ka.nnz[p] = nnz;
                ka.pool_off[p] = (int64_t)poff;
            }
        } else {
        // one block per pair. Software pipeline over the 32-row chunks: the row counts are
        // fetched two chunks ahead and a row's first entry group one chunk ahead, so that a chunk starts with its
        // loads already landed instead of paying two dependent L2 round trips.
        auto cnt_at = [&](int i) -> int { return i <= n ? __ldcg(rowcnt + i) : 0; };
        auto grp_at = [&](int i, int g, float4& lo, float4& hi) {
            const char* q = slot + (int64_t)(i + 32) * stride + g * 32;
            lo = ld_cg_f4(q);
            hi = ld_cg_f4(q + 16);
        };
        int running = 0;
        int c_cur = cnt_at(1 + lane), c_nxt = cnt_at(33 + lane);
        float4 lo = make_float4(0.f, 0.f, 0.f, 0.f), hi = lo;
        if (ok && c_cur > 0) grp_at(1 + lane, (c_cur - 1) >> 2, lo, hi);
        for (int i0 = 1; i0 <= n; i0 += 32) {
            const int i = i0 + lane;
            const bool valid = i <= n;
            const int c = c_cur;
            const int c_nn = cnt_at(i + 64);
            float4 lo_n = make_float4(0.f, 0.f, 0.f, 0.f), hi_n = lo_n;
            if (ok && c_nxt > 0) grp_at(i + 32, (c_nxt - 1) >> 2, lo_n, hi_n);
            const int ex = warp_excl_scan(c, lane);
            const int tot = __shfl_sync(kFull, ex + c, 31);
            int d = running + ex;
            if (valid) rp[i - 1] = d;
            running += tot;
            if (ok && valid) {
                const char* buf = slot + (int64_t)(i + 32) * stride;
                for (int g = (c - 1) >> 2; g >= 0; --g) {   // the next group's loads are in flight while this one is stored
                    float4 nlo = lo, nhi = hi;
                    if (g > 0) {
                        nlo = ld_cg_f4(buf + (g - 1) * 32);
                        nhi = ld_cg_f4(buf + (g - 1) * 32 + 16);
                    }
                    const int q = 4 * g;
                    if (q + 3 < c) { pool[d] = make_float2(hi.z, hi.w); ++d; }
                    if (q + 2 < c) { pool[d] = make_float2(hi.x, hi.y); ++d; }
                    if (q + 1 < c) { pool[d] = make_float2(lo.z, lo.w); ++d; }
                    pool[d] = make_float2(lo.x, lo.y); ++d;
                    lo = nlo;
                    hi = nhi;
                }
            }
            c_cur = c_nxt;
            c_nxt = c_nn;
            lo = lo_n;
            hi = hi_n;
        }
        if (lane == 0) {
            rp[n] = running;
            ka.nnz[p] = nnz;
            ka.pool_off[p] = (int64_t)poff;
        }
        }
    }

    // ---- memory-limited mode only: histogram of the kept values over the threshold bins -------------
    // A second walk over the entry buffers, so that the emission above stays as it is for every other call.
    if constexpr (kCsr) {
        if (ka.tau_hist != nullptr) {   // warp-uniform
            const int32_t* rowcnt = (const int32_t*)(slot + rowcnt_offset(n, C, nb, RB));
            for (int i = 1 + 32 * warp + lane; i <= n; i += 32 * W)
                for (int b = 0; b < nb; ++b) {
                    const int cb = __ldcg(rowcnt + (int64_t)b * (n + 1) + i);
                    const float2* buf = (const float2*)(slot + (int64_t)b * blk_bytes + (int64_t)(i + 32) * stride);
                    for (int e = 0; e < cb; ++e) {
                        const int bin = (__float_as_int(__ldcg(&buf[e].x)) - ka.tau_bits0) >> kTauShift;
                        atomicAdd(&hist_s[min(max(bin, 0), kTauBins - 1)], 1u);
                    }
                }
        }
    }
}

}  // namespace qp
