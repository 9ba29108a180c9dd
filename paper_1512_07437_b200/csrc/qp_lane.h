// qp_lane.h -- per-lane arithmetic of the striped wavefront DP (forward, backward, combine, MEA, sparsify).
//
// One warp processes one sequence pair. The DP grid is the extended (n+1) x (m+1) grid of SURVEY.md 8(c) c-1
// (row 0 / column 0 included; a sentinel residue code with zero match emission makes M vanish there).
// Lane l owns C consecutive columns of a 32*C-column block and processes row i = t - l at step t, so a lane
// needs (a) its own previous-row values (registers), (b) the boundary values of the lane on its left
// (forward) or right (backward), handed over by warp shuffle in the caller (qp_pair.cuh).
//
// Number representation ("block floating point"): every lane keeps its DP values as R-typed mantissas times
// 2^e with a per-lane, per-model integer exponent e. Path weights are plain probabilities (linear space), the
// exponent carries the log2 scale. Rescaling multiplies by exact powers of two, so it adds no rounding error.
// This replaces the paper-lineage log-sum-exp arithmetic: same posterior (the method's result is exact, the
// oracle is its definition), ~8x fewer instructions, no transcendental per cell, and ~100x smaller error than
// fp32 log-space.
//
// Recurrences (linear-space restatement of SURVEY.md 8(c) c-1, after the background normalisation of pin 8:
// em(a,b) = exp(lm[a][b]-lx[a]-lx[b]), insert emissions = 1):
//   forward   S(i,j)   = wMM*M(i,j) + sum_g wIM_g*(X_g(i,j)+Y_g(i,j))      (everything that can enter M(i+1,j+1))
//             M(i,j)   = em(x_i,y_j) * S(i-1,j-1)
//             X_g(i,j) = wMI_g*M(i-1,j) + wII_g*X_g(i-1,j)
//             Y_g(i,j) = wMI_g*M(i,j-1) + wII_g*Y_g(i,j-1)
//   backward  T(i,j)   = em(x_{i+1},y_{j+1}) * BM(i+1,j+1)
//             BM(i,j)  = wMM*T(i,j) + sum_g wMI_g*(BX_g(i+1,j) + BY_g(i,j+1))
//             BX_g(i,j)= wIM_g*T(i,j) + wII_g*BX_g(i+1,j)
//             BY_g(i,j)= wIM_g*T(i,j) + wII_g*BY_g(i,j+1)
//   start/end weights are injected at cells (0,0),(0,1) and (n,m) in the SPECIAL step variants.
//
// This header is plain C++ (no CUDA intrinsics) so that tests/simt_emu can compile the very same lane code
// for the host and step 32 emulated lanes in lockstep. It contains no oracle code and the oracle none of this.
#pragma once
#include <math.h>
#include <stdint.h>
#include <string.h>

#if defined(__CUDACC__)
#define QP_HD __host__ __device__ __forceinline__
#else
#define QP_HD inline
#endif

namespace qp {

constexpr int kSentinel = 31;   // residue code with zero match emission (row 0, column 0, padding)
constexpr int kTabDim = 32;     // emission table is kTabDim x kTabDim
constexpr int kMaxIns = 2;
constexpr int kZeroExp = -100000;  // "exponent" of 0

template <typename R> struct Traits;
template <> struct Traits<float> {
    using acc_t = int32_t;               // MEA fixed-point accumulator
    struct alignas(8) vec2 { float x, y; };
    static constexpr int kMaxShift = 127;
};
template <> struct Traits<double> {
    using acc_t = int64_t;
    struct alignas(16) vec2 { double x, y; };
    static constexpr int kMaxShift = 1023;
};

// 2^e; e below the normal range gives exactly 0, above it is clamped (callers flag that case)
QP_HD float pow2i(int e, float) {
    e = e < -127 ? -127 : (e > 127 ? 127 : e);
    uint32_t b = (uint32_t)(e + 127) << 23;
    float f;
    memcpy(&f, &b, 4);
    return f;
}
QP_HD double pow2i(int e, double) {
    e = e < -1023 ? -1023 : (e > 1023 ? 1023 : e);
    uint64_t b = (uint64_t)(e + 1023) << 52;
    double f;
    memcpy(&f, &b, 8);
    return f;
}
// floor(log2 v) for normal v > 0; kZeroExp for 0 / denormal
QP_HD int expo(float v) {
    uint32_t b;
    memcpy(&b, &v, 4);
    int e = (int)((b >> 23) & 0xff);
    return e == 0 ? kZeroExp : e - 127;
}
QP_HD int expo(double v) {
    uint64_t b;
    memcpy(&b, &v, 8);
    int e = (int)((b >> 52) & 0x7ff);
    return e == 0 ? kZeroExp : e - 1023;
}
QP_HD float qfma(float a, float b, float c) { return fmaf(a, b, c); }
QP_HD double qfma(double a, double b, double c) { return fma(a, b, c); }
QP_HD float qmax(float a, float b) { return fmaxf(a, b); }
QP_HD double qmax(double a, double b) { return fmax(a, b); }
QP_HD int imax(int a, int b) { return a > b ? a : b; }

// linear-space weights of one model; unused insert slots are 0
template <typename R> struct Weights {
    R wMM, wMI[kMaxIns], wII[kMaxIns], wIM[kMaxIns];
    R initM, initI[kMaxIns], endM, endI[kMaxIns];
};

// ---------------------------------------------------------------------------------------------------------
// forward
// ---------------------------------------------------------------------------------------------------------
template <typename R, int G> struct FwdEx {   // a lane's last column of the row it just finished
    R S, M, Y[G];
    int e;
};
template <typename R, int G> struct FwdRun {  // values carried along a row
    R Sdiag, Ml, Yl[G];
    R mwl[G];        // wMI[g] * M(i, j-1): shared by X_g(i+1, j-1) and Y_g(i, j)
};
struct FwdSpecial {      // which injections/captures apply to this lane in a SPECIAL step
    bool start;          // lane holds cell (0,0) and is at row 0: inject init weights at k=0 / k=1
    bool capture;        // lane holds cell (n,m) and is at row n: capture Z at k = kz
    int kz;
};

template <typename R, int G, int C> struct FwdModel {
    R S[C];          // S(i-1, j) for own columns (becomes the diagonal input of the next row)
    R Xn[G][C];      // X_g(i, j) for the row about to be computed
    R Sdin;          // S(i-1, j0-1): left neighbour's S of the previous row, already at exponent e
    int e;
    R f1, f2;        // cached scale factor of the incoming values: 2^(rin.e - e) = f1 * f2 (f2 != 1 only if rare)
    bool rare;
    FwdEx<R, G> ex;

    QP_HD void init() {
        for (int k = 0; k < C; ++k) {
            S[k] = R(0);
            for (int g = 0; g < G; ++g) Xn[g][k] = R(0);
        }
        Sdin = R(0);
        e = 0;
        f1 = f2 = R(1);
        rare = false;
        ex.S = ex.M = R(0);
        for (int g = 0; g < G; ++g) ex.Y[g] = R(0);
        ex.e = 0;
    }

    // Scale bookkeeping, called only on the steps where a scale can change (warp-uniform decision of the caller):
    //   first       this lane is on its first row (i == 0): its own values are still all zero, so it only has to pick
    //               the exponent that normalises the values that come in (lane-divergent, a handful of instructions);
    //   rescale_now periodic renormalisation (warp-uniform): looks at the own values AND the incoming ones, so
    //               nothing leaves the range before the next renormalisation;
    //   recompute   the cached factor 2^(rin.e - e) = f1 * f2 is rebuilt (renormalisation step and the step after it:
    //               that is when this lane's or its neighbour's exponent changes).
    // zero_in: nothing comes in (first lane of the first block): the incoming values count as 0.
    QP_HD void prepare(const FwdEx<R, G>& rin, bool first, bool rescale_now, bool recompute, bool zero_in,
                       int& range_flag) {
        if (first) {   // own values are all zero: take the scale that normalises what comes in
            f1 = R(0);
            f2 = R(1);
            rare = false;
            if (!zero_in) {
                R mi = qmax(rin.S, rin.M);
#pragma unroll
                for (int g = 0; g < G; ++g) mi = qmax(mi, rin.Y[g]);
                int ki = expo(mi);
                ki = ki == kZeroExp ? 0 : ki;
                e = rin.e + ki;
                f1 = pow2i(-ki, R(0));
            }
        }
        if (recompute) {
            if (rescale_now) {
                R mo = Sdin;
                R mi = qmax(rin.S, rin.M);
#pragma unroll
                for (int k = 0; k < C; ++k) {
                    mo = qmax(mo, S[k]);
#pragma unroll
                    for (int g = 0; g < G; ++g) mo = qmax(mo, Xn[g][k]);
                }
#pragma unroll
                for (int g = 0; g < G; ++g) mi = qmax(mi, rin.Y[g]);
                int ko = expo(mo), ki = zero_in ? kZeroExp : expo(mi);
                ki = ki == kZeroExp ? kZeroExp : ki + (rin.e - e);
                int k = imax(ko, ki);
                if (k != kZeroExp && k != 0) {
                    R f = pow2i(-k, R(0));
#pragma unroll
                    for (int c = 0; c < C; ++c) {
                        S[c] *= f;
#pragma unroll
                        for (int g = 0; g < G; ++g) Xn[g][c] *= f;
                    }
                    Sdin *= f;
                    e += k;
                }
            }
            const int d = rin.e - e;
            f2 = R(1);
            rare = false;
            if (zero_in) {
                f1 = R(0);
            } else if (d <= 60) {
                f1 = pow2i(d, R(0));
            } else {
                // rare: large exponent gap (e.g. a lane that has not renormalised yet). Scale in two exact steps;
                // only a value that would really leave the range is an error.
                R mi = qmax(rin.S, rin.M);
#pragma unroll
                for (int g = 0; g < G; ++g) mi = qmax(mi, rin.Y[g]);
                const int ki = expo(mi);
                int dd = d;
                if (ki != kZeroExp && ki + d > Traits<R>::kMaxShift - 27) {
                    range_flag = 1;
                    dd = Traits<R>::kMaxShift - 27 - ki;
                }
                f1 = pow2i(dd >> 1, R(0));
                f2 = pow2i(dd - (dd >> 1), R(0));
                rare = true;
            }
        }
    }

    // every step: bring the neighbour's values to the own scale. any_rare (warp-uniform): some lane of the warp
    // needs the second factor.
    QP_HD void load(const FwdEx<R, G>& rin, bool any_rare, FwdRun<R, G>& run, const Weights<R>& w) {
        run.Sdiag = Sdin;
        run.Ml = rin.M * f1;
        Sdin = rin.S * f1;
#pragma unroll
        for (int g = 0; g < G; ++g) run.Yl[g] = rin.Y[g] * f1;
        if (any_rare) {
            run.Ml *= f2;
            Sdin *= f2;
#pragma unroll
            for (int g = 0; g < G; ++g) run.Yl[g] *= f2;
        }
#pragma unroll
        for (int g = 0; g < G; ++g) run.mwl[g] = w.wMI[g] * run.Ml;
    }

    // one cell; returns M(i,j) (at exponent e). SPECIAL adds the start injection / Z capture.
    template <bool SPECIAL>
    QP_HD R cell(int k, R em, FwdRun<R, G>& run, const Weights<R>& w, const FwdSpecial& sp, R& zcap) {
        R M = em * run.Sdiag;
        run.Sdiag = S[k];
        R acc = R(0), zacc = R(0);
#pragma unroll
        for (int g = 0; g < G; ++g) {
            R X = Xn[g][k];
            R Y = qfma(w.wII[g], run.Yl[g], run.mwl[g]);            // the row chain runs through one FMA only
            if (SPECIAL && sp.start && k == 1) Y = w.initI[g];      // Y_g(0,1) = init_I[g]
            R xy = X + Y;
            acc = g == 0 ? w.wIM[g] * xy : qfma(w.wIM[g], xy, acc);
            if (SPECIAL) zacc = qfma(w.endI[g], xy, zacc);
            const R mw = w.wMI[g] * M;                              // used by X_g(i+1,j) now and Y_g(i,j+1) next
            Xn[g][k] = qfma(w.wII[g], X, mw);
            run.mwl[g] = mw;
            run.Yl[g] = Y;
        }
        R Sn = qfma(w.wMM, M, acc);   // small terms first, dominant term last: one rounding at full magnitude
        if (SPECIAL && sp.start && k == 0) {                          // cell (0,0): the start state
            Sn = w.initM;                                             //   -> M(1,1) = em * init_M
#pragma unroll
            for (int g = 0; g < G; ++g) Xn[g][k] = w.initI[g];        //   -> X_g(1,0) = init_I[g]
        }
        if (SPECIAL && sp.capture && k == sp.kz) zcap = qfma(w.endM, M, zacc);   // Z = sum_s end_s F_s(n,m)
        S[k] = Sn;
        run.Ml = M;
        return M;
    }

    QP_HD void end(const FwdRun<R, G>& run) {
        ex.S = S[C - 1];
        ex.M = run.Ml;
#pragma unroll
        for (int g = 0; g < G; ++g) ex.Y[g] = run.Yl[g];
        ex.e = e;
    }
};

// ---------------------------------------------------------------------------------------------------------
// backward
// ---------------------------------------------------------------------------------------------------------
template <typename R, int G> struct BwdEx {   // a lane's first column of the row it just finished
    R TL, BY[G];     // TL = em(x_i,y_j0)*BM(i,j0) = T(i-1, j0-1)
    int e;
};
template <typename R, int G> struct BwdRun {
    R Tc, BYr[G];
};
struct BwdSpecial {
    bool end;        // lane holds cell (n,m) and is at row n: inject end weights at k = kz
    bool capture;    // lane holds cell (0,0) and is at row 0: capture Z_b at k = 0
    int kz;
};

template <typename R, int G, int C> struct BwdModel {
    R Tn[C];         // T(i, j) for the row about to be computed
    R BXn[G][C];     // BX_g(i+1, j)
    int e;
    R f1, f2;        // cached scale factor of the incoming values (FwdModel)
    bool rare;
    BwdEx<R, G> ex;

    QP_HD void init() {
        for (int k = 0; k < C; ++k) {
            Tn[k] = R(0);
            for (int g = 0; g < G; ++g) BXn[g][k] = R(0);
        }
        e = 0;
        f1 = f2 = R(1);
        rare = false;
        ex.TL = R(0);
        for (int g = 0; g < G; ++g) ex.BY[g] = R(0);
        ex.e = 0;
    }

    // see FwdModel::prepare; first: the lane is on row n; zero_in: last lane of the last block
    QP_HD void prepare(const BwdEx<R, G>& rin, bool first, bool rescale_now, bool recompute, bool zero_in,
                       int& range_flag) {
        if (first) {   // own values are all zero: take the scale that normalises what comes in
            f1 = R(0);
            f2 = R(1);
            rare = false;
            if (!zero_in) {
                R mi = rin.TL;
#pragma unroll
                for (int g = 0; g < G; ++g) mi = qmax(mi, rin.BY[g]);
                int ki = expo(mi);
                ki = ki == kZeroExp ? 0 : ki;
                e = rin.e + ki;
                f1 = pow2i(-ki, R(0));
            }
        }
        if (recompute) {
            if (rescale_now) {
                R mo = R(0);
                R mi = rin.TL;
#pragma unroll
                for (int k = 0; k < C; ++k) {
                    mo = qmax(mo, Tn[k]);
#pragma unroll
                    for (int g = 0; g < G; ++g) mo = qmax(mo, BXn[g][k]);
                }
#pragma unroll
                for (int g = 0; g < G; ++g) mi = qmax(mi, rin.BY[g]);
                int ko = expo(mo), ki = zero_in ? kZeroExp : expo(mi);
                ki = ki == kZeroExp ? kZeroExp : ki + (rin.e - e);
                int k = imax(ko, ki);
                if (k != kZeroExp && k != 0) {
                    R f = pow2i(-k, R(0));
#pragma unroll
                    for (int c = 0; c < C; ++c) {
                        Tn[c] *= f;
#pragma unroll
                        for (int g = 0; g < G; ++g) BXn[g][c] *= f;
                    }
                    e += k;
                }
            }
            const int d = rin.e - e;
            f2 = R(1);
            rare = false;
            if (zero_in) {
                f1 = R(0);
            } else if (d <= 60) {
                f1 = pow2i(d, R(0));
            } else {   // rare, see FwdModel::prepare
                R mi = rin.TL;
#pragma unroll
                for (int g = 0; g < G; ++g) mi = qmax(mi, rin.BY[g]);
                const int ki = expo(mi);
                int dd = d;
                if (ki != kZeroExp && ki + d > Traits<R>::kMaxShift - 27) {
                    range_flag = 1;
                    dd = Traits<R>::kMaxShift - 27 - ki;
                }
                f1 = pow2i(dd >> 1, R(0));
                f2 = pow2i(dd - (dd >> 1), R(0));
                rare = true;
            }
        }
    }

    QP_HD void load(const BwdEx<R, G>& rin, bool any_rare, BwdRun<R, G>& run) {
        run.Tc = rin.TL * f1;
#pragma unroll
        for (int g = 0; g < G; ++g) run.BYr[g] = rin.BY[g] * f1;
        if (any_rare) {
            run.Tc *= f2;
#pragma unroll
            for (int g = 0; g < G; ++g) run.BYr[g] *= f2;
        }
    }

    // one cell (columns are walked right to left); returns BM(i,j) at exponent e
    template <bool SPECIAL>
    QP_HD R cell(int k, R em, BwdRun<R, G>& run, const Weights<R>& w, const BwdSpecial& sp, R& zcap) {
        R T = Tn[k];
        Tn[k] = run.Tc;             // T(i-1, j): produced by the cell on the right, consumed one row later
        R acc = R(0), zacc = R(0);
#pragma unroll
        for (int g = 0; g < G; ++g) {
            R bx = BXn[g][k];
            R s = bx + run.BYr[g];
            acc = g == 0 ? w.wMI[g] * s : qfma(w.wMI[g], s, acc);
            if (SPECIAL) zacc = qfma(w.initI[g], s, zacc);
            const R tw = w.wIM[g] * T;                               // enters both BX_g(i,j) and BY_g(i,j)
            BXn[g][k] = qfma(w.wII[g], bx, tw);
            run.BYr[g] = qfma(w.wII[g], run.BYr[g], tw);             // row chain: one FMA per cell
        }
        R BM = qfma(w.wMM, T, acc);
        if (SPECIAL && sp.end && k == sp.kz) {                        // cell (n,m): B_s(n,m) = end_s
            BM = w.endM;
#pragma unroll
            for (int g = 0; g < G; ++g) {
                BXn[g][k] = w.endI[g];
                run.BYr[g] = w.endI[g];
            }
        }
        // Z_b = init_M*em(x1,y1)*BM(1,1) + sum_g init_I[g]*(BX_g(1,0) + BY_g(0,1)), all visible at cell (0,0)
        if (SPECIAL && sp.capture && k == 0) zcap = qfma(w.initM, T, zacc);
        run.Tc = em * BM;
        return BM;
    }

    QP_HD void end(const BwdRun<R, G>& run) {
        ex.TL = run.Tc;
#pragma unroll
        for (int g = 0; g < G; ++g) ex.BY[g] = run.BYr[g];
        ex.e = e;
    }
};

// ---------------------------------------------------------------------------------------------------------
// combine + MEA quantisation
// ---------------------------------------------------------------------------------------------------------
// P_model * sqrt(1/2) = (F*B) * c with c = 2^E * sqrt(1/2)/Zm, E = eF + eB - eZ. The product F*B of two mantissas
// cannot overflow (each stays below 2^57 between renormalisations) and 0 * c is 0, so no NaN can arise. A large positive
// E means that every cell of the lane's stripe has a tiny F*B (F peaks at one end of the stripe, B at the other: long
// gaps through a wide stripe, e.g. 1029 x 489 unrelated residues in the C = 16 class). F*B = P * Zm * 2^-E is still a
// normal number of full precision while P >= 2^(E - 126) (fp32) and flushes to zero below, so up to kMaxE = 96 every
// posterior above 2^-30 is exact and the rest is zero to working precision; beyond kMaxE the caller reports a range
// error instead of computing inexactly. (Round 1 had kMaxE = 64 for fp32: a random-model fuzz with rows >> columns
// tripped it on posteriors that are perfectly representable.)
template <typename R> struct PScale {
    static constexpr int kMaxE = sizeof(R) == 4 ? 96 : 512;
    R c;
    QP_HD bool set(int E, R invZr) {
        const bool bad = E > kMaxE;
        E = E > kMaxE ? kMaxE : E;
        c = pow2i(E, R(0)) * invZr;   // pow2i clamps below: 2^E -> 0, the posterior is 0 to working precision
        return bad;
    }
    QP_HD R apply(R F, R B) const { return (F * B) * c; }
};
// 1/Zm with the sqrt(1/2) of the root mean square folded in
template <typename R> QP_HD R inv_z_rms(R Zm) { return R(0.70710678118654752440) / Zm; }

QP_HD float qsqrt(float v) {
#if defined(__CUDA_ARCH__)
    float r;
    asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(v));
    return r;
#else
    return sqrtf(v);
#endif
}
QP_HD double qsqrt(double v) { return sqrt(v); }

// P = sqrt((P_hmm^2 + P_pf^2)/2); the arguments already carry the factor sqrt(1/2) (PScale)
template <typename R> QP_HD R combine_rms(R ph, R pp) { return qsqrt(qfma(ph, ph, pp * pp)); }

// MEA fixed point: q = round(P * 2^s). fp32: magic-constant rounding (valid while P*2^s < 2^22)
QP_HD int32_t quantise(float p, float scale) {
    float t = fmaf(p, scale, 12582912.0f);
    int32_t b;
    memcpy(&b, &t, 4);
    return b - 0x4B400000;
}
QP_HD int64_t quantise(double p, double scale) { return (int64_t)llrint(p * scale); }

}  // namespace qp
