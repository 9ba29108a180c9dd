// qp_both.cuh -- the two automata of one lane side by side (pair-HMM with G = 2 insert-state pairs + partition
// function with GP), behind one interface for the wavefront driver (qp_pair.cuh).
//
//   FwdBoth<R,GP,C> / BwdBoth<R,GP,C>   generic: the two scalar models of qp_lane.h next to each other.
//   FwdBoth<float,1,C> / BwdBoth<float,1,C>   the production case (fp32, one insert-state pair in the partition
//       function): the M / X_1 / Y_1 recurrences of the two automata have the same shape, so their values are kept
//       as (hmm, pf) register pairs and updated with Blackwell's packed fp32 instructions (PTX fma/mul/add.rn.f32x2
//       -> SASS FFMA2/FMUL2/FADD2: one issue slot, two IEEE-rounded results, measured at the full 128 FMA/clk/SM).
//       The pair-HMM's second insert-state pair stays scalar. The emission table entry (em_hmm, em_pf) and the stored
//       F word (F_hmm, F_pf) are such pairs already. Every result is bit-identical to the scalar formulation (same
//       operations, same order, each rounded once), which is what tests/simt_emu steps on the CPU.
// The kernel is issue-bound, so halving the issue slots of ~2/3 of the arithmetic is the point.
#pragma once
#include "qp_lane.h"

namespace qp {

// paired weights (hmm, pf) of the part the two automata share in shape (insert-state pair 0) + the pair-HMM's second
// pair; filled on the host (qp_api.cu) and passed in the kernel argument block, so that the packed instructions can
// take them as 64-bit constant-bank operands
struct alignas(8) W2 {
    Traits<float>::vec2 MM, MI, II, IM, initI, endI, initM, endM;
    float MI1, II1, IM1, initI1, endI1, pad_;
    void set(const Weights<float>& h, const Weights<float>& p) {
        MM = {h.wMM, p.wMM};
        MI = {h.wMI[0], p.wMI[0]};
        II = {h.wII[0], p.wII[0]};
        IM = {h.wIM[0], p.wIM[0]};
        initI = {h.initI[0], p.initI[0]};
        endI = {h.endI[0], p.endI[0]};
        initM = {h.initM, p.initM};
        endM = {h.endM, p.endM};
        MI1 = h.wMI[1];
        II1 = h.wII[1];
        IM1 = h.wIM[1];
        initI1 = h.initI[1];
        endI1 = h.endI[1];
        pad_ = 0.f;
    }
};

// ------------------------------------------------------------------------------------------------------------
// generic: two scalar models
// ------------------------------------------------------------------------------------------------------------
template <typename R, int GP, int C> struct FwdBoth {
    using V2 = typename Traits<R>::vec2;
    FwdModel<R, 2, C> H;
    FwdModel<R, GP, C> P;
    FwdRun<R, 2> rH;
    FwdRun<R, GP> rP;
    __device__ __forceinline__ void init() { H.init(); P.init(); }
    __device__ __forceinline__ void prepare(const FwdEx<R, 2>& rh, const FwdEx<R, GP>& rp, bool first, bool resc,
                                            bool recompute, bool zero_in, int& range_flag) {
        H.prepare(rh, first, resc, recompute, zero_in, range_flag);
        P.prepare(rp, first, resc, recompute, zero_in, range_flag);
    }
    __device__ __forceinline__ bool rare_h() const { return H.rare; }
    __device__ __forceinline__ bool rare_p() const { return P.rare; }
    __device__ __forceinline__ void load(const FwdEx<R, 2>& rh, const FwdEx<R, GP>& rp, bool any_h, bool any_p,
                                         const Weights<R>& wh, const Weights<R>& wp, const W2&) {
        H.load(rh, any_h, rH, wh);
        P.load(rp, any_p, rP, wp);
    }
    template <bool S>
    __device__ __forceinline__ V2 cell(int k, V2 em, const Weights<R>& wh, const Weights<R>& wp, const W2&,
                                       const FwdSpecial& sp, R& zcap_h, R& zcap_p) {
        V2 o;
        o.x = H.template cell<S>(k, em.x, rH, wh, sp, zcap_h);
        o.y = P.template cell<S>(k, em.y, rP, wp, sp, zcap_p);
        return o;
    }
    __device__ __forceinline__ void end() { H.end(rH); P.end(rP); }
    __device__ __forceinline__ const FwdEx<R, 2>& exh() const { return H.ex; }
    __device__ __forceinline__ const FwdEx<R, GP>& exp() const { return P.ex; }
    __device__ __forceinline__ int eh() const { return H.e; }
    __device__ __forceinline__ int ep() const { return P.e; }
};

template <typename R, int GP, int C> struct BwdBoth {
    using V2 = typename Traits<R>::vec2;
    BwdModel<R, 2, C> H;
    BwdModel<R, GP, C> P;
    BwdRun<R, 2> rH;
    BwdRun<R, GP> rP;
    __device__ __forceinline__ void init() { H.init(); P.init(); }
    __device__ __forceinline__ void prepare(const BwdEx<R, 2>& rh, const BwdEx<R, GP>& rp, bool first, bool resc,
                                            bool recompute, bool zero_in, int& range_flag) {
        H.prepare(rh, first, resc, recompute, zero_in, range_flag);
        P.prepare(rp, first, resc, recompute, zero_in, range_flag);
    }
    __device__ __forceinline__ bool rare_h() const { return H.rare; }
    __device__ __forceinline__ bool rare_p() const { return P.rare; }
    __device__ __forceinline__ void load(const BwdEx<R, 2>& rh, const BwdEx<R, GP>& rp, bool any_h, bool any_p) {
        H.load(rh, any_h, rH);
        P.load(rp, any_p, rP);
    }
    // returns (BM_hmm, BM_pf); zh / zp receive the backward totals on the capturing cell
    template <bool S>
    __device__ __forceinline__ V2 cell(int k, V2 em, const Weights<R>& wh, const Weights<R>& wp, const W2&,
                                       const BwdSpecial& sp, R& zh, R& zp) {
        V2 o;
        o.x = H.template cell<S>(k, em.x, rH, wh, sp, zh);
        o.y = P.template cell<S>(k, em.y, rP, wp, sp, zp);
        return o;
    }
    // (P_hmm, P_pf) * sqrt(1/2) of one cell
    __device__ __forceinline__ V2 posterior(V2 F, V2 B, const PScale<R>& psh, const PScale<R>& psp) const {
        V2 o;
        o.x = psh.apply(F.x, B.x);
        o.y = psp.apply(F.y, B.y);
        return o;
    }
    __device__ __forceinline__ void end() { H.end(rH); P.end(rP); }
    __device__ __forceinline__ const BwdEx<R, 2>& exh() const { return H.ex; }
    __device__ __forceinline__ const BwdEx<R, GP>& exp() const { return P.ex; }
    __device__ __forceinline__ int eh() const { return H.e; }
    __device__ __forceinline__ int ep() const { return P.e; }
};

// ------------------------------------------------------------------------------------------------------------
// packed fp32 pairs
// ------------------------------------------------------------------------------------------------------------
using F2 = Traits<float>::vec2;   // (hmm, pf)

__device__ __forceinline__ unsigned long long f2_bits(F2 a) {
    unsigned long long r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(a.x), "f"(a.y));
    return r;
}
__device__ __forceinline__ F2 f2_from(unsigned long long b) {
    F2 r;
    asm("mov.b64 {%0, %1}, %2;" : "=f"(r.x), "=f"(r.y) : "l"(b));
    return r;
}
__device__ __forceinline__ F2 f2(float x, float y) {
    F2 r;
    r.x = x;
    r.y = y;
    return r;
}
__device__ __forceinline__ F2 f2_fma(F2 a, F2 b, F2 c) {
    unsigned long long r;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(f2_bits(a)), "l"(f2_bits(b)), "l"(f2_bits(c)));
    return f2_from(r);
}
__device__ __forceinline__ F2 f2_mul(F2 a, F2 b) {
    unsigned long long r;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(f2_bits(a)), "l"(f2_bits(b)));
    return f2_from(r);
}
__device__ __forceinline__ F2 f2_add(F2 a, F2 b) {
    unsigned long long r;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(f2_bits(a)), "l"(f2_bits(b)));
    return f2_from(r);
}

// scale bookkeeping of one model on the packed state: the same decisions as FwdModel/BwdModel::prepare, written
// once for a component selector (0 = hmm, 1 = pf)
struct Scale {
    int e;
    float f1, f2;
    bool rare;
    __device__ __forceinline__ void init() {
        e = 0;
        f1 = f2 = 1.f;
        rare = false;
    }
    // first row: pick the exponent that normalises the incoming maximum `mi`
    __device__ __forceinline__ void adopt(float mi, int rin_e, bool zero_in) {
        f1 = 0.f;
        f2 = 1.f;
        rare = false;
        if (!zero_in) {
            int ki = expo(mi);
            ki = ki == kZeroExp ? 0 : ki;
            e = rin_e + ki;
            f1 = pow2i(-ki, 0.f);
        }
    }
    // renormalisation shift for own maximum `mo` and incoming maximum `mi`: returns k (0: nothing to do)
    __device__ __forceinline__ int shift(float mo, float mi, int rin_e, bool zero_in) const {
        int ko = expo(mo), ki = zero_in ? kZeroExp : expo(mi);
        ki = ki == kZeroExp ? kZeroExp : ki + (rin_e - e);
        const int k = imax(ko, ki);
        return k == kZeroExp ? 0 : k;
    }
    __device__ __forceinline__ void factors(float mi, int rin_e, bool zero_in, int& range_flag) {
        const int d = rin_e - e;
        f2 = 1.f;
        rare = false;
        if (zero_in) {
            f1 = 0.f;
        } else if (d <= 60) {
            f1 = pow2i(d, 0.f);
        } else {   // rare, see FwdModel::prepare
            const int ki = expo(mi);
            int dd = d;
            if (ki != kZeroExp && ki + d > Traits<float>::kMaxShift - 27) {
                range_flag = 1;
                dd = Traits<float>::kMaxShift - 27 - ki;
            }
            f1 = pow2i(dd >> 1, 0.f);
            f2 = pow2i(dd - (dd >> 1), 0.f);
            rare = true;
        }
    }
};

template <int C> struct FwdBoth<float, 1, C> {
    using V2 = F2;
    F2 S[C], X0[C], Sdin;     // (hmm, pf): S(i-1,j), X_1(i,j), S(i-1,j0-1)
    float X1[C];              // pair-HMM X_2(i,j)
    Scale sh, sp;
    FwdEx<float, 2> xh;
    FwdEx<float, 1> xp;
    F2 Sdiag, Ml, Yl0, mwl0;  // values carried along a row
    float Yl1, mwl1;

    __device__ __forceinline__ void init() {
#pragma unroll
        for (int k = 0; k < C; ++k) {
            S[k] = X0[k] = f2(0.f, 0.f);
            X1[k] = 0.f;
        }
        Sdin = f2(0.f, 0.f);
        sh.init();
        sp.init();
        xh.S = xh.M = xh.Y[0] = xh.Y[1] = 0.f;
        xp.S = xp.M = xp.Y[0] = 0.f;
        xh.e = xp.e = 0;
    }
    __device__ __forceinline__ void prepare(const FwdEx<float, 2>& rh, const FwdEx<float, 1>& rp, bool first, bool resc,
                                            bool recompute, bool zero_in, int& range_flag) {
        const float mi_h = fmaxf(fmaxf(rh.S, rh.M), fmaxf(rh.Y[0], rh.Y[1])), mi_p = fmaxf(fmaxf(rp.S, rp.M), rp.Y[0]);
        if (first) {
            sh.adopt(mi_h, rh.e, zero_in);
            sp.adopt(mi_p, rp.e, zero_in);
        }
        if (recompute) {
            if (resc) {
                float mo_h = Sdin.x, mo_p = Sdin.y;
#pragma unroll
                for (int k = 0; k < C; ++k) {
                    mo_h = fmaxf(mo_h, fmaxf(fmaxf(S[k].x, X0[k].x), X1[k]));
                    mo_p = fmaxf(mo_p, fmaxf(S[k].y, X0[k].y));
                }
                const int kh = sh.shift(mo_h, mi_h, rh.e, zero_in), kp = sp.shift(mo_p, mi_p, rp.e, zero_in);
                if ((kh | kp) != 0) {
                    const F2 f = f2(pow2i(-kh, 0.f), pow2i(-kp, 0.f));
#pragma unroll
                    for (int k = 0; k < C; ++k) {
                        S[k] = f2_mul(S[k], f);
                        X0[k] = f2_mul(X0[k], f);
                        X1[k] *= f.x;
                    }
                    Sdin = f2_mul(Sdin, f);
                    sh.e += kh;
                    sp.e += kp;
                }
            }
            sh.factors(mi_h, rh.e, zero_in, range_flag);
            sp.factors(mi_p, rp.e, zero_in, range_flag);
        }
    }
    __device__ __forceinline__ bool rare_h() const { return sh.rare; }
    __device__ __forceinline__ bool rare_p() const { return sp.rare; }
    __device__ __forceinline__ void load(const FwdEx<float, 2>& rh, const FwdEx<float, 1>& rp, bool any_h, bool any_p,
                                         const Weights<float>&, const Weights<float>&, const W2& w) {
        Sdiag = Sdin;
        Ml = f2(rh.M * sh.f1, rp.M * sp.f1);
        Sdin = f2(rh.S * sh.f1, rp.S * sp.f1);
        Yl0 = f2(rh.Y[0] * sh.f1, rp.Y[0] * sp.f1);
        Yl1 = rh.Y[1] * sh.f1;
        if (any_h) {
            Ml.x *= sh.f2;
            Sdin.x *= sh.f2;
            Yl0.x *= sh.f2;
            Yl1 *= sh.f2;
        }
        if (any_p) {
            Ml.y *= sp.f2;
            Sdin.y *= sp.f2;
            Yl0.y *= sp.f2;
        }
        mwl0 = f2_mul(w.MI, Ml);
        mwl1 = w.MI1 * Ml.x;
    }
    template <bool SPEC>
    __device__ __forceinline__ F2 cell(int k, F2 em, const Weights<float>&, const Weights<float>&, const W2& w,
                                       const FwdSpecial& sp_, float& zcap_h, float& zcap_p) {
        const F2 M = f2_mul(em, Sdiag);
        Sdiag = S[k];
        F2 Y0 = f2_fma(w.II, Yl0, mwl0);
        float Y1 = fmaf(w.II1, Yl1, mwl1);
        if (SPEC && sp_.start && k == 1) {   // Y_g(0,1) = init_I[g]
            Y0 = w.initI;
            Y1 = w.initI1;
        }
        const F2 xy0 = f2_add(X0[k], Y0);
        const float xy1 = X1[k] + Y1;
        F2 acc = f2_mul(w.IM, xy0);
        acc.x = fmaf(w.IM1, xy1, acc.x);
        const F2 mw0 = f2_mul(w.MI, M);
        const float mw1 = w.MI1 * M.x;
        X0[k] = f2_fma(w.II, X0[k], mw0);
        X1[k] = fmaf(w.II1, X1[k], mw1);
        mwl0 = mw0;
        mwl1 = mw1;
        Yl0 = Y0;
        Yl1 = Y1;
        F2 Sn = f2_fma(w.MM, M, acc);
        if (SPEC && sp_.start && k == 0) {   // cell (0,0): the start state
            Sn = w.initM;
            X0[k] = w.initI;
            X1[k] = w.initI1;
        }
        if (SPEC && sp_.capture && k == sp_.kz) {   // Z = sum_s end_s F_s(n,m)
            F2 zacc = f2_mul(w.endI, xy0);
            zacc.x = fmaf(w.endI1, xy1, zacc.x);
            const F2 z = f2_fma(w.endM, M, zacc);
            zcap_h = z.x;
            zcap_p = z.y;
        }
        S[k] = Sn;
        Ml = M;
        return M;
    }
    __device__ __forceinline__ void end() {
        xh.S = S[C - 1].x;
        xh.M = Ml.x;
        xh.Y[0] = Yl0.x;
        xh.Y[1] = Yl1;
        xh.e = sh.e;
        xp.S = S[C - 1].y;
        xp.M = Ml.y;
        xp.Y[0] = Yl0.y;
        xp.e = sp.e;
    }
    __device__ __forceinline__ const FwdEx<float, 2>& exh() const { return xh; }
    __device__ __forceinline__ const FwdEx<float, 1>& exp() const { return xp; }
    __device__ __forceinline__ int eh() const { return sh.e; }
    __device__ __forceinline__ int ep() const { return sp.e; }
};

template <int C> struct BwdBoth<float, 1, C> {
    using V2 = F2;
    F2 Tn[C], BX0[C];         // (hmm, pf): T(i,j), BX_1(i+1,j)
    float BX1[C];             // pair-HMM BX_2(i+1,j)
    Scale sh, sp;
    BwdEx<float, 2> xh;
    BwdEx<float, 1> xp;
    F2 Tc, BYr0;
    float BYr1;

    __device__ __forceinline__ void init() {
#pragma unroll
        for (int k = 0; k < C; ++k) {
            Tn[k] = BX0[k] = f2(0.f, 0.f);
            BX1[k] = 0.f;
        }
        sh.init();
        sp.init();
        xh.TL = xh.BY[0] = xh.BY[1] = 0.f;
        xp.TL = xp.BY[0] = 0.f;
        xh.e = xp.e = 0;
    }
    __device__ __forceinline__ void prepare(const BwdEx<float, 2>& rh, const BwdEx<float, 1>& rp, bool first, bool resc,
                                            bool recompute, bool zero_in, int& range_flag) {
        const float mi_h = fmaxf(rh.TL, fmaxf(rh.BY[0], rh.BY[1])), mi_p = fmaxf(rp.TL, rp.BY[0]);
        if (first) {
            sh.adopt(mi_h, rh.e, zero_in);
            sp.adopt(mi_p, rp.e, zero_in);
        }
        if (recompute) {
            if (resc) {
                float mo_h = 0.f, mo_p = 0.f;
#pragma unroll
                for (int k = 0; k < C; ++k) {
                    mo_h = fmaxf(mo_h, fmaxf(fmaxf(Tn[k].x, BX0[k].x), BX1[k]));
                    mo_p = fmaxf(mo_p, fmaxf(Tn[k].y, BX0[k].y));
                }
                const int kh = sh.shift(mo_h, mi_h, rh.e, zero_in), kp = sp.shift(mo_p, mi_p, rp.e, zero_in);
                if ((kh | kp) != 0) {
                    const F2 f = f2(pow2i(-kh, 0.f), pow2i(-kp, 0.f));
#pragma unroll
                    for (int k = 0; k < C; ++k) {
                        Tn[k] = f2_mul(Tn[k], f);
                        BX0[k] = f2_mul(BX0[k], f);
                        BX1[k] *= f.x;
                    }
                    sh.e += kh;
                    sp.e += kp;
                }
            }
            sh.factors(mi_h, rh.e, zero_in, range_flag);
            sp.factors(mi_p, rp.e, zero_in, range_flag);
        }
    }
    __device__ __forceinline__ bool rare_h() const { return sh.rare; }
    __device__ __forceinline__ bool rare_p() const { return sp.rare; }
    __device__ __forceinline__ void load(const BwdEx<float, 2>& rh, const BwdEx<float, 1>& rp, bool any_h, bool any_p) {
        Tc = f2(rh.TL * sh.f1, rp.TL * sp.f1);
        BYr0 = f2(rh.BY[0] * sh.f1, rp.BY[0] * sp.f1);
        BYr1 = rh.BY[1] * sh.f1;
        if (any_h) {
            Tc.x *= sh.f2;
            BYr0.x *= sh.f2;
            BYr1 *= sh.f2;
        }
        if (any_p) {
            Tc.y *= sp.f2;
            BYr0.y *= sp.f2;
        }
    }
    template <bool SPEC>
    __device__ __forceinline__ F2 cell(int k, F2 em, const Weights<float>&, const Weights<float>&, const W2& w,
                                       const BwdSpecial& sp_, float& zh, float& zp) {
        const F2 T = Tn[k];
        Tn[k] = Tc;   // T(i-1, j): produced by the cell on the right, consumed one row later
        const F2 s0 = f2_add(BX0[k], BYr0);
        const float s1 = BX1[k] + BYr1;
        F2 acc = f2_mul(w.MI, s0);
        acc.x = fmaf(w.MI1, s1, acc.x);
        const F2 tw0 = f2_mul(w.IM, T);
        const float tw1 = w.IM1 * T.x;
        BX0[k] = f2_fma(w.II, BX0[k], tw0);
        BX1[k] = fmaf(w.II1, BX1[k], tw1);
        BYr0 = f2_fma(w.II, BYr0, tw0);
        BYr1 = fmaf(w.II1, BYr1, tw1);
        F2 BM = f2_fma(w.MM, T, acc);
        if (SPEC && sp_.end && k == sp_.kz) {   // cell (n,m): B_s(n,m) = end_s
            BM = w.endM;
            BX0[k] = w.endI;
            BX1[k] = w.endI1;
            BYr0 = w.endI;
            BYr1 = w.endI1;
        }
        if (SPEC && sp_.capture && k == 0) {    // Z_b, all of it visible at cell (0,0)
            F2 zacc = f2_mul(w.initI, s0);
            zacc.x = fmaf(w.initI1, s1, zacc.x);
            const F2 z = f2_fma(w.initM, T, zacc);
            zh = z.x;
            zp = z.y;
        }
        Tc = f2_mul(em, BM);
        return BM;
    }
    __device__ __forceinline__ F2 posterior(F2 F, F2 B, const PScale<float>& psh, const PScale<float>& psp) const {
        return f2_mul(f2_mul(F, B), f2(psh.c, psp.c));
    }
    __device__ __forceinline__ void end() {
        xh.TL = Tc.x;
        xh.BY[0] = BYr0.x;
        xh.BY[1] = BYr1;
        xh.e = sh.e;
        xp.TL = Tc.y;
        xp.BY[0] = BYr0.y;
        xp.e = sp.e;
    }
    __device__ __forceinline__ const BwdEx<float, 2>& exh() const { return xh; }
    __device__ __forceinline__ const BwdEx<float, 1>& exp() const { return xp; }
    __device__ __forceinline__ int eh() const { return sh.e; }
    __device__ __forceinline__ int ep() const { return sp.e; }
};

}  // namespace qp
