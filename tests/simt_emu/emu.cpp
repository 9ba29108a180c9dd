// emu.cpp -- TEST HARNESS (CPU): steps 32 emulated lanes in lockstep through the lane arithmetic of the CUDA
// path (paper_1512_07437_b200/csrc/qp_lane.h, compiled here for the host). It mirrors the wavefront driver of
// qp_pair.cuh (who processes which row when, what is handed to the neighbour, where the start/end weights are
// injected) so the kernel's logic can be checked against the oracle on a box without a GPU. It is NOT a product
// path: nothing in the package links or loads it, and it contains no oracle code.
#include <cmath>
#include <cstdint>
#include <cstdlib>
#include <cstring>
#include <vector>

#include "qp_lane.h"

using namespace qp;

struct EmuModel {   // linear weights + 32x32 emission table (already background-normalised), doubles
    double em[32 * 32];
    double wMM, wMI[2], wII[2], wIM[2], initM, initI[2], endM, endI[2];
};

template <typename R> static Weights<R> to_w(const EmuModel& m) {
    Weights<R> w;
    w.wMM = (R)m.wMM; w.initM = (R)m.initM; w.endM = (R)m.endM;
    for (int g = 0; g < 2; ++g) { w.wMI[g] = (R)m.wMI[g]; w.wII[g] = (R)m.wII[g]; w.wIM[g] = (R)m.wIM[g]; w.initI[g] = (R)m.initI[g]; w.endI[g] = (R)m.endI[g]; }
    return w;
}

struct Kept { int row, col; float val; };

template <typename R, int GP, int C>
static int emu_pair(const EmuModel& mh, const EmuModel& mp, const uint8_t* xs, int n, const uint8_t* ys, int m, double tau,
                    int mask, float* dense /*n*m*/, double* logZ2 /*4: log2 Zf_h, Zb_h, Zf_p, Zb_p (normalised model)*/,
                    double* dist, std::vector<Kept>& csr, std::vector<int>& row_ptr) {
    using Acc = typename Traits<R>::acc_t;
    struct V2 { R x, y; };
    const Weights<R> wh = to_w<R>(mh), wp = to_w<R>(mp);
    const int nb = (m + 1 + 32 * C - 1) / (32 * C);
    const int T = n + 32;
    const int cols_last = (m + 1) - (nb - 1) * 32 * C;
    const int lz = (cols_last - 1) / C, kz = (cols_last - 1) % C;
    std::vector<V2> F((size_t)nb * T * C * 32);
    std::vector<int> EH((size_t)nb * T * 32), EP((size_t)nb * T * 32);
    auto Fat = [&](int b, int t, int k, int lane) -> V2& { return F[(((size_t)b * T + t) * C + (C - 1 - k)) * 32 + lane]; };
    std::vector<FwdEx<R, 2>> bndH(n + 1), bndHn(n + 1);
    std::vector<FwdEx<R, GP>> bndP(n + 1), bndPn(n + 1);
    int range_flag = 0;
    R zcap_h = 0, zcap_p = 0; int ez_h = 0, ez_p = 0;
    // ---------------- forward
    for (int b = 0; b < nb; ++b) {
        std::vector<FwdModel<R, 2, C>> H(32); std::vector<FwdModel<R, GP, C>> Pm(32);
        for (int l = 0; l < 32; ++l) { H[l].init(); Pm[l].init(); }
        const bool last = b == nb - 1;
        const int tend = n + (last ? lz : 31);
        bool any_rare_h = false, any_rare_p = false;
        for (int t = 0; t <= tend; ++t) {
            FwdEx<R, 2> rh[32]; FwdEx<R, GP> rp[32];
            for (int l = 0; l < 32; ++l) {
                int i = t - l; bool active = i >= 0 && i <= n;
                if (l > 0) { rh[l] = H[l - 1].ex; rp[l] = Pm[l - 1].ex; }
                else if (b > 0 && active) { rh[0] = bndH[i]; rp[0] = bndP[i]; }
                else { rh[0] = H[0].ex; rp[0] = Pm[0].ex; }   // shfl_up leaves lane 0 its own value; zero_in makes it count as 0
            }
            const bool special = (b == 0 && t == 0) || (last && t == tend);
            // qp_pair.cuh, all warp-uniform: ramp = lanes are entering their first row; recompute = a scale can change
            const bool ramp = t < 32, recompute = (t & mask) <= 1 || (b > 0 && t > n), prep = ramp || recompute;
            const bool resc = (t & mask) == 0;
            if (prep) {
                any_rare_h = any_rare_p = false;
                for (int l = 0; l < 32; ++l) {
                    int i = t - l; bool active = i >= 0 && i <= n;
                    const bool zin = l == 0 && !(b > 0 && active);
                    H[l].prepare(rh[l], i == 0, resc, recompute, zin, range_flag); Pm[l].prepare(rp[l], i == 0, resc, recompute, zin, range_flag);
                    any_rare_h |= H[l].rare; any_rare_p |= Pm[l].rare;
                }
            }
            for (int l = 0; l < 32; ++l) {
                int i = t - l; bool active = i >= 0 && i <= n;
                int xcode = (i >= 1 && i <= n) ? xs[i - 1] : kSentinel;
                FwdRun<R, 2> runH; FwdRun<R, GP> runP;
                FwdEx<R, 2> qh = rh[l]; FwdEx<R, GP> qp_ = rp[l];
                if (!prep) { qh.e = 123456; qp_.e = -123456; }   // the kernel does not shuffle the exponents then
                H[l].load(qh, any_rare_h, runH, wh); Pm[l].load(qp_, any_rare_p, runP, wp);
                FwdSpecial sp; sp.start = special && (b == 0 && l == 0 && i == 0); sp.capture = special && (last && l == lz && i == n); sp.kz = kz;
                for (int k = 0; k < C; ++k) {
                    int j = b * 32 * C + l * C + k;
                    int ycode = (j >= 1 && j <= m) ? ys[j - 1] : kSentinel;
                    R eh = (R)mh.em[xcode * 32 + ycode], ep = (R)mp.em[xcode * 32 + ycode];
                    V2 o; R dz = 0;
                    if (special) { o.x = H[l].template cell<true>(k, eh, runH, wh, sp, zcap_h); o.y = Pm[l].template cell<true>(k, ep, runP, wp, sp, zcap_p); }
                    else { o.x = H[l].template cell<false>(k, eh, runH, wh, sp, dz); o.y = Pm[l].template cell<false>(k, ep, runP, wp, sp, dz); }
                    if (active) Fat(b, t, k, l) = o;
                }
                H[l].end(runH); Pm[l].end(runP);
                if (active) { EH[((size_t)b * T + t) * 32 + l] = H[l].e; EP[((size_t)b * T + t) * 32 + l] = Pm[l].e;
                    if (!last && l == 31) { bndHn[i] = H[l].ex; bndPn[i] = Pm[l].ex; } }
            }
        }
        if (last) { ez_h = H[lz].e; ez_p = Pm[lz].e; }
        bndH.swap(bndHn); bndP.swap(bndPn);
    }
    { int kh = expo(zcap_h), kp = expo(zcap_p);
      if (kh == kZeroExp || kp == kZeroExp) return -8;
      zcap_h *= pow2i(-kh, R(0)); zcap_p *= pow2i(-kp, R(0)); ez_h += kh; ez_p += kp; }
    const R invZh = inv_z_rms(zcap_h), invZp = inv_z_rms(zcap_p);
    // ---------------- backward
    const int minnm = n < m ? n : m;
    int sbits = (int)(8 * sizeof(Acc)) - 2; { int need = 1; while ((1 << need) <= minnm) ++need; sbits -= need; int cap = sizeof(R) == 4 ? 20 : 40; if (sbits > cap) sbits = cap; }
    const R mea_scale = (R)ldexp(1.0, sbits);
    std::vector<BwdEx<R, 2>> bH(n + 1), bHn(n + 1); std::vector<BwdEx<R, GP>> bP(n + 1), bPn(n + 1); std::vector<Acc> bA(n + 1), bAn(n + 1);
    std::vector<std::vector<Kept>> parked((size_t)nb * T * 32);   // entries parked per (block, step, lane), in arrival order
    R zb_h = 0, zb_p = 0; int ezb_h = 0, ezb_p = 0; Acc mea = 0;
    for (int b = nb - 1; b >= 0; --b) {
        std::vector<BwdModel<R, 2, C>> H(32); std::vector<BwdModel<R, GP, C>> Pm(32);
        std::vector<std::vector<Acc>> An(32, std::vector<Acc>(C, 0)); std::vector<Acc> Adin(32, 0), exA(32, 0);
        for (int l = 0; l < 32; ++l) { H[l].init(); Pm[l].init(); }
        const bool last = b == nb - 1; const int tstart = n + (last ? lz : 31);
        bool any_rare_h = false, any_rare_p = false;
        for (int t = tstart; t >= 0; --t) {
            BwdEx<R, 2> rh[32]; BwdEx<R, GP> rp[32]; Acc rA[32];
            for (int l = 0; l < 32; ++l) {
                int i = t - l; bool active = i >= 0 && i <= n;
                if (l < 31) { rh[l] = H[l + 1].ex; rp[l] = Pm[l + 1].ex; rA[l] = exA[l + 1]; }
                else if (!last && active) { rh[l] = bH[i]; rp[l] = bP[i]; rA[l] = bA[i]; }
                else { rh[l] = H[l].ex; rp[l] = Pm[l].ex; rA[l] = 0; }   // shfl_down leaves lane 31 its own value
            }
            const bool special = (last && t == tstart) || (b == 0 && t == 0);
            const bool ramp = t >= n, recompute = (t & mask) >= mask - 1 || (!last && t < 32), prep = ramp || recompute;
            const bool resc = (t & mask) == mask;
            if (prep) {
                any_rare_h = any_rare_p = false;
                for (int l = 0; l < 32; ++l) {
                    int i = t - l; bool active = i >= 0 && i <= n;
                    const bool zin = l == 31 && !(!last && active);
                    H[l].prepare(rh[l], i == n, resc, recompute, zin, range_flag); Pm[l].prepare(rp[l], i == n, resc, recompute, zin, range_flag);
                    any_rare_h |= H[l].rare; any_rare_p |= Pm[l].rare;
                }
            }
            for (int l = 0; l < 32; ++l) {
                int i = t - l; bool active = i >= 0 && i <= n;
                int xcode = (i >= 1 && i <= n) ? xs[i - 1] : kSentinel;
                BwdRun<R, 2> runH; BwdRun<R, GP> runP;
                BwdEx<R, 2> qh = rh[l]; BwdEx<R, GP> qp_ = rp[l];
                if (!prep) { qh.e = 123456; qp_.e = -123456; }
                H[l].load(qh, any_rare_h, runH); Pm[l].load(qp_, any_rare_p, runP);
                int eFh = active ? EH[((size_t)b * T + t) * 32 + l] : 0, eFp = active ? EP[((size_t)b * T + t) * 32 + l] : 0;
                PScale<R> psh, psp;
                if ((psh.set(eFh + H[l].e - ez_h, invZh) | psp.set(eFp + Pm[l].e - ez_p, invZp)) && active && b * 32 * C + l * C <= m) range_flag = 1;
                Acc Adiag = Adin[l], Aright = rA[l];
                BwdSpecial sp; sp.end = special && (last && l == lz && i == n); sp.capture = special && (b == 0 && l == 0 && i == 0); sp.kz = kz;
                for (int k = C - 1; k >= 0; --k) {
                    int j = b * 32 * C + l * C + k;
                    int ycode = (j >= 1 && j <= m) ? ys[j - 1] : kSentinel;
                    R eh = (R)mh.em[xcode * 32 + ycode], ep = (R)mp.em[xcode * 32 + ycode];
                    R zh = 0, zp = 0, bmh, bmp;
                    if (special) { bmh = H[l].template cell<true>(k, eh, runH, wh, sp, zh); bmp = Pm[l].template cell<true>(k, ep, runP, wp, sp, zp); }
                    else { bmh = H[l].template cell<false>(k, eh, runH, wh, sp, zh); bmp = Pm[l].template cell<false>(k, ep, runP, wp, sp, zp); }
                    if (special && sp.capture && k == 0) { zb_h = zh; zb_p = zp; ezb_h = H[l].e; ezb_p = Pm[l].e; }
                    V2 f; if (active) f = Fat(b, t, k, l); else { f.x = 0; f.y = 0; }
                    R ph = psh.apply(f.x, bmh), pp = psp.apply(f.y, bmp);
                    R P = combine_rms(ph, pp);
                    Acc q = quantise(P, mea_scale);
                    Acc a = Adiag + q; a = a > An[l][k] ? a : An[l][k]; a = a > Aright ? a : Aright;
                    Adiag = An[l][k]; An[l][k] = a; Aright = a;
                    if (P >= (R)tau) parked[((size_t)b * T + t) * 32 + l].push_back({i - 1, j - 1, (float)P});
                    if (dense && i >= 1 && i <= n && j >= 1 && j <= m) dense[(size_t)(i - 1) * m + (j - 1)] = (float)P;
                }
                H[l].end(runH); Pm[l].end(runP);
                exA[l] = An[l][0]; Adin[l] = rA[l];
                if (active && b > 0 && l == 0) { bHn[i] = H[l].ex; bPn[i] = Pm[l].ex; bAn[i] = exA[l]; }
            }
        }
        if (b == 0) mea = An[0][0];
        bH.swap(bHn); bP.swap(bPn); bA.swap(bAn);
    }
    *dist = 1.0 - (double)mea / (ldexp(1.0, sbits) * (double)minnm);
    logZ2[0] = std::log2((double)zcap_h) + ez_h; logZ2[1] = std::log2((double)zb_h) + ezb_h;
    logZ2[2] = std::log2((double)zcap_p) + ez_p; logZ2[3] = std::log2((double)zb_p) + ezb_p;
    // ---------------- CSR traversal order of qp_pair.cuh: rows ascending; within a row blocks, lanes ascending;
    // inside a (step,lane) the parked entries reversed
    csr.clear(); row_ptr.assign(n + 1, 0);
    for (int i = 1; i <= n; ++i) {
        row_ptr[i - 1] = (int)csr.size();
        for (int b = 0; b < nb; ++b)
            for (int l = 0; l < 32; ++l) {
                if (b * 32 * C + l * C > m) continue;
                auto& v = parked[((size_t)b * T + (i + l)) * 32 + l];
                for (int e = (int)v.size() - 1; e >= 0; --e) csr.push_back(v[e]);
            }
    }
    row_ptr[n] = (int)csr.size();
    return range_flag ? -8 : 0;
}

static std::vector<Kept> g_csr; static std::vector<int> g_rp;

extern "C" int emu_run(int fp64, int GP, int C, const EmuModel* mh, const EmuModel* mp, const uint8_t* xs, int n, const uint8_t* ys,
                       int m, double tau, int mask, float* dense, double* logZ2, double* dist) {
#define RUN(R, G, CC) return emu_pair<R, G, CC>(*mh, *mp, xs, n, ys, m, tau, mask, dense, logZ2, dist, g_csr, g_rp)
    if (!fp64 && GP == 1) { switch (C) { case 2: RUN(float, 1, 2); case 3: RUN(float, 1, 3); case 4: RUN(float, 1, 4); case 8: RUN(float, 1, 8); case 9: RUN(float, 1, 9); case 10: RUN(float, 1, 10); case 16: RUN(float, 1, 16); } }
    if (!fp64 && GP == 2) { switch (C) { case 2: RUN(float, 2, 2); case 6: RUN(float, 2, 6); } }
    if (fp64 && GP == 2) { switch (C) { case 2: RUN(double, 2, 2); case 4: RUN(double, 2, 4); case 8: RUN(double, 2, 8); } }
    return -1;
}
extern "C" int emu_csr_nnz() { return (int)g_csr.size(); }
extern "C" void emu_csr_get(int* row_ptr, int* rows, int* cols, float* vals) {
    for (size_t q = 0; q < g_rp.size(); ++q) row_ptr[q] = g_rp[q];
    for (size_t q = 0; q < g_csr.size(); ++q) { rows[q] = g_csr[q].row; cols[q] = g_csr[q].col; vals[q] = g_csr[q].val; }
}
