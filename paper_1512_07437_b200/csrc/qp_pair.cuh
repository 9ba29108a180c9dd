// qp_pair.cuh -- one warp takes one sequence pair through the whole hot path:
//   forward (pair-HMM + partition function, fused)
//   backward (both models) fused with combine, sparsify, MEA  8(a) a2, a4, a5, a6, a7
//   warp-scan compaction of the kept entries into CSR         8(a) a6
// Lane arithmetic lives in qp_lane.h; this file owns the wavefront (who processes which row when), the warp
// shuffles that hand row boundaries to the neighbouring lane, and all global-memory traffic.
#pragma once
#include <cuda_runtime.h>

#include <type_traits>

#include "qp_internal.h"

namespace qp {

constexpr unsigned kFull = 0xffffffffu;

__device__ __forceinline__ float shfl_up1(float v) { return __shfl_up_sync(kFull, v, 1); }
__device__ __forceinline__ double shfl_up1(double v) { return __shfl_up_sync(kFull, v, 1); }
__device__ __forceinline__ int shfl_up1(int v) { return __shfl_up_sync(kFull, v, 1); }
__device__ __forceinline__ float shfl_dn1(float v) { return __shfl_down_sync(kFull, v, 1); }
__device__ __forceinline__ double shfl_dn1(double v) { return __shfl_down_sync(kFull, v, 1); }
__device__ __forceinline__ int shfl_dn1(int v) { return __shfl_down_sync(kFull, v, 1); }
__device__ __forceinline__ int64_t shfl_dn1(int64_t v) { return (int64_t)__shfl_down_sync(kFull, (long long)v, 1); }

template <typename R, int G> __device__ __forceinline__ FwdEx<R, G> shfl_up_ex(const FwdEx<R, G>& a) {
    FwdEx<R, G> r;
    r.S = shfl_up1(a.S);
    r.M = shfl_up1(a.M);
#pragma unroll
    for (int g = 0; g < G; ++g) r.Y[g] = shfl_up1(a.Y[g]);
    r.e = shfl_up1(a.e);
    return r;
}
template <typename R, int G> __device__ __forceinline__ BwdEx<R, G> shfl_dn_ex(const BwdEx<R, G>& a) {
    BwdEx<R, G> r;
    r.TL = shfl_dn1(a.TL);
#pragma unroll
    for (int g = 0; g < G; ++g) r.BY[g] = shfl_dn1(a.BY[g]);
    r.e = shfl_dn1(a.e);
    return r;
}
template <typename R, int G> __device__ __forceinline__ void zero_ex(FwdEx<R, G>& a) {
    a.S = a.M = R(0);
#pragma unroll
    for (int g = 0; g < G; ++g) a.Y[g] = R(0);
    a.e = 0;
}
template <typename R, int G> __device__ __forceinline__ void zero_ex(BwdEx<R, G>& a) {
    a.TL = R(0);
#pragma unroll
    for (int g = 0; g < G; ++g) a.BY[g] = R(0);
    a.e = 0;
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

struct alignas(8) Entry {   // a kept posterior, parked in the consumed forward slot of its (step, lane)
    float val;
    int32_t k;              // column offset inside the lane's stripe
};

// park a kept entry without a branch (predicated 8-byte store)
__device__ __forceinline__ void st_entry_if(void* ptr, float val, int k, bool keep) {
    asm volatile(
        "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %3, 0;\n\t@p st.global.v2.b32 [%0], {%1, %2};\n\t}"
        :
        : "l"(ptr), "r"(__float_as_int(val)), "r"(k), "r"((int)keep)
        : "memory");
}

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

// ---------------------------------------------------------------------------------------------------------
// the pair pipeline
// ---------------------------------------------------------------------------------------------------------
template <typename R, int GP, int C>
__device__ void process_pair(const KArgs<R>& ka, const typename Traits<R>::vec2* __restrict__ tab, int p, char* slot,
                             int lane) {
    using V2 = typename Traits<R>::vec2;
    using Acc = typename Traits<R>::acc_t;
    constexpr int RB = (int)sizeof(R);
    constexpr int GH = 2;

    const PairInfo pi = ka.info[p];
    const int n = pi.n, m = pi.m;
    const int nb = (m + 1 + 32 * C - 1) / (32 * C);   // column blocks (column 0 included)
    const uint8_t* __restrict__ xs = ka.seqs + pi.xoff;
    const uint8_t* __restrict__ ys = ka.seqs + pi.yoff;
    const int64_t stride = step_stride(C, RB);
    const int64_t blk_bytes = (int64_t)num_steps(n) * stride;
    const int cols_last = (m + 1) - (nb - 1) * 32 * C;   // columns (incl. column 0) that fall in the last block
    const int lz = (cols_last - 1) / C, kz = (cols_last - 1) % C;   // lane / stripe offset of column m
    const int mask = ka.rescale_mask;
    char* bnd0 = slot + (int64_t)nb * blk_bytes;
    char* bnd1 = bnd0 + (int64_t)(n + 1) * bnd_rec_bytes(RB);
    int range_flag = 0;
    auto xcode_at = [&](int i) -> int { return (i >= 1 && i <= n) ? (int)__ldg(xs + i - 1) : kSentinel; };

    // =========================================== forward ===================================================
    R zcap_h = R(0), zcap_p = R(0);
    int ez_h = 0, ez_p = 0;
    for (int b = 0; b < nb; ++b) {
        FwdModel<R, GH, C> H;
        FwdModel<R, GP, C> Pm;
        H.init();
        Pm.init();
        int ycode[C];
#pragma unroll
        for (int k = 0; k < C; ++k) {
            int j = b * 32 * C + lane * C + k;
            ycode[k] = (j >= 1 && j <= m) ? (int)ys[j - 1] : kSentinel;
        }
        char* blk = slot + (int64_t)b * blk_bytes;
        const bool last = (b == nb - 1);
        const int tend = n + (last ? lz : 31);
        const FwdBnd<R, GP>* bin = (const FwdBnd<R, GP>*)((b & 1) ? bnd0 : bnd1);   // written by block b-1
        FwdBnd<R, GP>* bout = (FwdBnd<R, GP>*)((b & 1) ? bnd1 : bnd0);
        int xnext = xcode_at(0 - lane);   // residue code of the row of the NEXT step, loaded one step ahead
        for (int t = 0; t <= tend; ++t) {
            const int i = t - lane;
            const bool active = (i >= 0) && (i <= n);
            const int xcode = xnext;
            xnext = xcode_at(i + 1);
            FwdEx<R, GH> rh = shfl_up_ex(H.ex);
            FwdEx<R, GP> rp = shfl_up_ex(Pm.ex);
            if (lane == 0) {
                if (b > 0 && active) {
                    const FwdBnd<R, GP> rec = ld_volatile(bin + i);
                    rh = rec.h;
                    rp = rec.p;
                } else {
                    zero_ex(rh);
                    zero_ex(rp);
                }
            }
            const bool resc = ((t & mask) == 0) || (i == 0);   // periodic, and on the lane's first row
            const V2* row = tab + xcode * kTabDim;
            V2* out = (V2*)(blk + (int64_t)t * stride);
            FwdRun<R, GH> runH;
            FwdRun<R, GP> runP;
            H.begin(rh, resc, runH, range_flag);
            Pm.begin(rp, resc, runP, range_flag);
            const bool special = (b == 0 && t == 0) || (last && t == tend);   // warp-uniform
            if (special) {
                FwdSpecial sp;
                sp.start = (b == 0 && lane == 0 && i == 0);
                sp.capture = (last && lane == lz && i == n);
                sp.kz = kz;
#pragma unroll
                for (int k = 0; k < C; ++k) {
                    V2 em = row[ycode[k]];
                    V2 o;
                    o.x = H.template cell<true>(k, em.x, runH, ka.wh, sp, zcap_h);
                    o.y = Pm.template cell<true>(k, em.y, runP, ka.wp, sp, zcap_p);
                    if (active) out[(C - 1 - k) * 32 + lane] = o;
                }
            } else {
                FwdSpecial sp;
                sp.start = sp.capture = false;
                sp.kz = 0;
                R dummy = R(0);
#pragma unroll
                for (int k = 0; k < C; ++k) {
                    V2 em = row[ycode[k]];
                    V2 o;
                    o.x = H.template cell<false>(k, em.x, runH, ka.wh, sp, dummy);
                    o.y = Pm.template cell<false>(k, em.y, runP, ka.wp, sp, dummy);
                    if (active) out[(C - 1 - k) * 32 + lane] = o;
                }
            }
            H.end(runH);
            Pm.end(runP);
            if (active) {
                int2 ee = make_int2(H.e, Pm.e);
                *(int2*)(blk + (int64_t)t * stride + exps_offset(C, RB) + lane * 8) = ee;
                if (nb > 1 && !last && lane == 31) {
                    bout[i].h = H.ex;
                    bout[i].p = Pm.ex;
                }
            }
        }
        if (last) {
            ez_h = H.e;
            ez_p = Pm.e;
        }
        if (nb > 1) __syncwarp();   // lane 31's boundary column must be visible to lane 0 of the next block
    }
    // Z = Zm * 2^eZ with Zm in [1,2); every lane gets a copy
    zcap_h = __shfl_sync(kFull, zcap_h, lz);
    zcap_p = __shfl_sync(kFull, zcap_p, lz);
    ez_h = __shfl_sync(kFull, ez_h, lz);
    ez_p = __shfl_sync(kFull, ez_p, lz);
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
    const R invZh = R(1) / zcap_h, invZp = R(1) / zcap_p;

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
    const bool want_csr = !ka.refine_pass;
    float* dense = (ka.dense_P != nullptr && want_csr) ? ka.dense_P + ka.dense_off[p] : nullptr;
    R zb_h = R(0), zb_p = R(0);
    int ezb_h = 0, ezb_p = 0;
    int nnz_lane = 0;
    Acc mea = 0;
    for (int b = nb - 1; b >= 0; --b) {
        BwdModel<R, GH, C> H;
        BwdModel<R, GP, C> Pm;
        H.init();
        Pm.init();
        Acc An[C];
        int ycode[C];
        unsigned jvalid = 0;
#pragma unroll
        for (int k = 0; k < C; ++k) {
            An[k] = 0;
            int j = b * 32 * C + lane * C + k;
            bool v = (j >= 1 && j <= m);
            ycode[k] = v ? (int)ys[j - 1] : kSentinel;
            jvalid |= (v ? 1u : 0u) << k;
        }
        Acc Adin = 0, exA = 0;
        char* blk = slot + (int64_t)b * blk_bytes;
        const bool last = (b == nb - 1);
        const int tstart = n + (last ? lz : 31);
        const BwdBnd<R, GP>* bin = (const BwdBnd<R, GP>*)((b & 1) ? bnd0 : bnd1);   // written by block b+1
        BwdBnd<R, GP>* bout = (BwdBnd<R, GP>*)((b & 1) ? bnd1 : bnd0);
        const int jbase = b * 32 * C + lane * C;
        int xnext = xcode_at(tstart - lane);
        // F values and exponents of a step are loaded one step ahead (at the end of the previous iteration)
        V2 Fv[C];
        int2 eF;
        auto load_step = [&](int t2) {
            const int i2 = t2 - lane;
            const bool act2 = (i2 >= 0) && (i2 <= n);
            const char* stp2 = blk + (int64_t)t2 * stride;
            const V2* in2 = (const V2*)stp2;
#pragma unroll
            for (int k = 0; k < C; ++k) {
                if (act2) Fv[k] = in2[(C - 1 - k) * 32 + lane];
                else { Fv[k].x = R(0); Fv[k].y = R(0); }
            }
            eF = act2 ? *(const int2*)(stp2 + exps_offset(C, RB) + lane * 8) : make_int2(0, 0);
        };
        load_step(tstart);
        for (int t = tstart; t >= 0; --t) {
            const int i = t - lane;
            const bool active = (i >= 0) && (i <= n);
            const int xcode = xnext;
            xnext = xcode_at(i - 1);
            char* stp = blk + (int64_t)t * stride;
            BwdEx<R, GH> rh = shfl_dn_ex(H.ex);
            BwdEx<R, GP> rp = shfl_dn_ex(Pm.ex);
            Acc rA = shfl_dn1(exA);
            if (lane == 31) {
                if (!last && active) {
                    const BwdBnd<R, GP> rec = ld_volatile(bin + i);
                    rh = rec.h;
                    rp = rec.p;
                    rA = rec.A;
                } else {
                    zero_ex(rh);
                    zero_ex(rp);
                    rA = 0;
                }
            }
            const bool resc = ((t & mask) == mask) || (i == n);
            const V2* row = tab + xcode * kTabDim;
            BwdRun<R, GH> runH;
            BwdRun<R, GP> runP;
            H.begin(rh, resc, runH, range_flag);
            Pm.begin(rp, resc, runP, range_flag);
            PScale<R> psh, psp;
            psh.set(eF.x + H.e - ez_h, invZh);
            psp.set(eF.y + Pm.e - ez_p, invZp);
            const bool special = (last && t == tstart) || (b == 0 && t == 0);   // warp-uniform
            BwdSpecial sp;
            sp.end = special && (last && lane == lz && i == n);
            sp.capture = special && (b == 0 && lane == 0 && i == 0);
            sp.kz = kz;
            // loop 1: the two backward recurrences; F(i,j) is replaced in place by the model posteriors
            auto rec_body = [&](auto SPEC, int k) {
                constexpr bool S = decltype(SPEC)::value;
                V2 em = row[ycode[k]];
                R zh = R(0), zp = R(0);
                R bmh = H.template cell<S>(k, em.x, runH, ka.wh, sp, zh);
                R bmp = Pm.template cell<S>(k, em.y, runP, ka.wp, sp, zp);
                if (S && sp.capture && k == 0) {
                    zb_h = zh;
                    zb_p = zp;
                    ezb_h = H.e;
                    ezb_p = Pm.e;
                }
                Fv[k].x = psh.apply(Fv[k].x, bmh);
                Fv[k].y = psp.apply(Fv[k].y, bmp);
            };
            if (special) {
#pragma unroll
                for (int k = C - 1; k >= 0; --k) rec_body(std::true_type{}, k);
            } else {
#pragma unroll
                for (int k = C - 1; k >= 0; --k) rec_body(std::false_type{}, k);
            }
            // loop 2: combine, expected-accuracy max-plus, threshold + parking of kept entries
            Acc Adiag = Adin, Aright = rA;
            int cnt = 0;
            char* park = stp + (int64_t)lane * sizeof(V2);
#pragma unroll
            for (int k = C - 1; k >= 0; --k) {
                const R P = combine_rms(Fv[k].x, Fv[k].y);
                const Acc q = quantise(P, mea_scale);
                Acc a = Adiag + q;
                a = a > An[k] ? a : An[k];
                a = a > Aright ? a : Aright;
                Adiag = An[k];
                An[k] = a;
                Aright = a;
                if (want_csr) {
                    const bool keep = P >= ka.tau;
                    st_entry_if(park, (float)P, k, keep);
                    park += keep ? 32 * (int)sizeof(V2) : 0;
                    cnt += keep ? 1 : 0;
                    if (dense != nullptr && i >= 1 && i <= n && ((jvalid >> k) & 1))
                        dense[(int64_t)(i - 1) * m + (jbase + k - 1)] = (float)P;
                }
            }
            if (t > 0) load_step(t - 1);
            H.end(runH);
            Pm.end(runP);
            exA = An[0];
            Adin = rA;
            if (active) {
                if (want_csr) *(uint8_t*)(stp + cnts_offset(C, RB) + lane) = (uint8_t)cnt;
                nnz_lane += cnt;
                if (nb > 1 && b > 0 && lane == 0) {
                    bout[i].h = H.ex;
                    bout[i].p = Pm.ex;
                    bout[i].A = exA;
                }
            }
        }
        if (b == 0) mea = An[0];   // lane 0 holds A'(0,0) = A(n,m)
        if (nb > 1) __syncwarp();
    }
    mea = __shfl_sync(kFull, mea, 0);
    const double dist = 1.0 - (double)mea / (ldexp(1.0, sbits) * (double)minnm);

    if (__any_sync(kFull, range_flag)) {
        if (lane == 0 && atomicCAS(&ka.hdr->status[0], 0, -8 /*QP_ERR_RANGE*/) == 0) ka.hdr->status[1] = p;
    }

    // ---- distance d = 1 - A(n,m)/min(n,m), both orientations; near-identical pairs are queued for fp64 --------
    if (lane == 0) {
        const int xi = ka.pairs[2 * (int64_t)p], yi = ka.pairs[2 * (int64_t)p + 1];
        ka.dist[(int64_t)xi * ka.k + yi] = (float)dist;
        ka.dist[(int64_t)yi * ka.k + xi] = (float)dist;
        if (!ka.refine_pass && (float)dist < ka.refine_below) {
            int nbd;
            const int c64 = choose_class(m + 1, ka.refine_cmask, &nbd);
            const int pos = atomicAdd(&ka.hdr->refine_count[c64], 1);
            ka.refine_list[(int64_t)c64 * ka.refine_stride + pos] = p;
            atomicMax(&ka.hdr->refine_slot_bytes[c64],
                      (unsigned long long)slot_bytes(n, 2 * (c64 + 1), nbd, 8));
        }
    }

    // ---- logZ (optional): undo the background normalisation, ln Z = ln2*(log2 Zm + eZ) + sum lx ---------
    if (ka.logZ != nullptr && want_csr) {
        double ch = 0.0, cp = 0.0;
        for (int q = lane; q < n; q += 32) { ch += ka.lx_h[xs[q]]; cp += ka.lx_p[xs[q]]; }
        for (int q = lane; q < m; q += 32) { ch += ka.lx_h[ys[q]]; cp += ka.lx_p[ys[q]]; }
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

    // ---- CSR: warp-scan compaction of the parked entries, rows ascending, columns ascending ---------------
    // Row i's entries sit at (step i+l, lane l) for l = 0..31 and blocks 0..nb-1: ascending (block, lane) is
    // ascending column; inside a lane they were parked right-to-left, so they are read back reversed.
    if (want_csr) {
        const int nnz = warp_sum(nnz_lane);
        unsigned long long poff = 0;
        if (lane == 0) poff = atomicAdd(&ka.hdr->pool_cursor, (unsigned long long)nnz);
        poff = __shfl_sync(kFull, poff, 0);
        const bool ok = (long long)(poff + (unsigned long long)nnz) <= (long long)ka.pool_cap;
        if (!ok && lane == 0) {
            if (atomicCAS(&ka.hdr->status[0], 0, -6 /*QP_ERR_NNZ_CAPACITY*/) == 0) ka.hdr->status[1] = p;
        }
        int32_t* rp = ka.row_ptr + ka.pair_row_base[p];
        int running = 0;
        // Segments (row i, block b) in row-major order, SEG at a time so that the loads of a batch are
        // independent: (1) the SEG count bytes, (2) SEG warp scans, (3) e-th entry of every segment, stores.
        constexpr int SEGM = 8;    // multi-block batch
        const int32_t colbase = lane * C - 1;
        if (nb == 1) {
            constexpr int SEG = 8;   // rows per batch (larger batches cost registers in the DP loops: measured slower)
            const char* base = slot + (int64_t)(1 + lane) * stride;          // row 1
            const char* cbase = base + cnts_offset(C, RB) + lane;
            const bool lane_in = colbase < m;                                 // lane owns at least one real column
            int cnx[SEG];   // counts of the NEXT batch, loaded while the current one is compacted
#pragma unroll
            for (int u = 0; u < SEG; ++u) cnx[u] = (lane_in && u < n) ? (int)*(const uint8_t*)(cbase + (int64_t)u * stride) : 0;
            for (int r0 = 0; r0 < n; r0 += SEG) {
                int cn[SEG], st[SEG];
#pragma unroll
                for (int u = 0; u < SEG; ++u) {
                    cn[u] = cnx[u];
                    const int rn = r0 + SEG + u;
                    cnx[u] = (lane_in && rn < n) ? (int)*(const uint8_t*)(cbase + (int64_t)rn * stride) : 0;
                }
                int maxc = 0;
#pragma unroll
                for (int u = 0; u < SEG; ++u) {
                    if (lane == 0 && r0 + u < n) rp[r0 + u] = running;
                    const int ex = warp_excl_scan(cn[u], lane);
                    st[u] = running + ex + cn[u] - 1;   // destination of this lane's FIRST parked entry (highest column)
                    running += __shfl_sync(kFull, ex + cn[u], 31);
                    maxc = cn[u] > maxc ? cn[u] : maxc;
                }
                if (ok) {
                    maxc = __reduce_max_sync(kFull, maxc);
                    const char* eb = base + (int64_t)r0 * stride + (int64_t)lane * sizeof(V2);
                    for (int e = 0; e < maxc; ++e) {
                        Entry en[SEG];
#pragma unroll
                        for (int u = 0; u < SEG; ++u)
                            if (e < cn[u]) en[u] = *(const Entry*)(eb + (int64_t)u * stride + (int64_t)e * 32 * sizeof(V2));
#pragma unroll
                        for (int u = 0; u < SEG; ++u)
                            if (e < cn[u]) {
                                const long long dst = (long long)poff + st[u] - e;
                                ka.pool_col[dst] = colbase + en[u].k;
                                ka.pool_val[dst] = en[u].val;
                            }
                    }
                }
            }
        } else {
            // segments (row i, block b) in row-major order
            const int nseg = n * nb;
            for (int s0 = 0; s0 < nseg; s0 += SEGM) {
                int cn[SEGM], st[SEGM];
                const char* sp[SEGM];
                int32_t jb[SEGM];
#pragma unroll
                for (int u = 0; u < SEGM; ++u) {
                    const int sg = s0 + u;
                    const int i = 1 + sg / nb, b = sg - (i - 1) * nb;
                    jb[u] = b * 32 * C + colbase;
                    sp[u] = slot + (int64_t)b * blk_bytes + (int64_t)(i + lane) * stride;
                    cn[u] = (sg < nseg && jb[u] < m) ? (int)*(const uint8_t*)(sp[u] + cnts_offset(C, RB) + lane) : 0;
                }
                int maxc = 0;
#pragma unroll
                for (int u = 0; u < SEGM; ++u) {
                    const int sg = s0 + u;
                    if (lane == 0 && sg < nseg && sg % nb == 0) rp[sg / nb] = running;
                    const int ex = warp_excl_scan(cn[u], lane);
                    st[u] = running + ex + cn[u] - 1;
                    running += __shfl_sync(kFull, ex + cn[u], 31);
                    maxc = cn[u] > maxc ? cn[u] : maxc;
                }
                if (ok) {
                    maxc = __reduce_max_sync(kFull, maxc);
                    for (int e = 0; e < maxc; ++e) {
                        Entry en[SEGM];
#pragma unroll
                        for (int u = 0; u < SEGM; ++u)
                            if (e < cn[u]) en[u] = *(const Entry*)(sp[u] + ((int64_t)e * 32 + lane) * sizeof(V2));
#pragma unroll
                        for (int u = 0; u < SEGM; ++u)
                            if (e < cn[u]) {
                                const long long dst = (long long)poff + st[u] - e;
                                ka.pool_col[dst] = jb[u] + en[u].k;
                                ka.pool_val[dst] = en[u].val;
                            }
                    }
                }
            }
        }
        if (lane == 0) {
            rp[n] = running;
            ka.nnz[p] = nnz;
            ka.pool_off[p] = (int64_t)poff;
        }
    }
}

}  // namespace qp
