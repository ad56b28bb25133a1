// sb_tiled.cuh -- the register-tiled node-weight kernel (sm_100a), fp32, forward and gradient.
//
// Same sums per evaluation as sb_kernels.cuh / sb_hoist.cuh, with
// the band integral re-associated as in sb_hoist.cuh (an exact exchange of two finite sums):
//     raw_o = sum_l At[l] * R_o[l],   At[l] = sum_j ew_j w_{l-i_j}(tau_j)   (NODE WEIGHTS of (unit, band)),
//     R_o[l] = sum_k wp_k(o) (M0 + x1 M1)[rb_o + k][l]                      (phase-collapsed row of o),
// ew_j = exp(c CL(lambda_j/(1+z))) W_j, w = Keys a = -1/2 weights (reading G1).
//
// What differs from sb_hoist.cuh is WHO holds WHAT.  There a lane reloaded the four phase rows of
// {M0, M1} for every observation (four LDG.64 per eight FFMA: bound by the L1 data pipe).  Here a CTA
// works on a GROUP of up to 32 units that are neighbours in redshift (stable z-order, sb_hoist.cuh),
// in ROUNDS of at most `cap` observations.  Per round: the observations are counting-sorted in shared
// memory by (band, first phase row rb); the geometry of every (band, unit) item and the union node
// window of every band are computed by all threads; then, one STAGE (a set of bands) at a time, two
// phases separated by a CTA barrier:
//   phase A  one warp per ITEM (unit, band): lanes own model cells of the band's common node grid,
//            walk the band samples of their cell (colour factor x folded weight, moments sum ew tau^p),
//            turn the moments into node weights and store At[item][node] in SHARED MEMORY (512 nodes
//            per item and window segment; wider windows take several segments);
//   phase B  the observations of a band, sorted by rb, are cut into equal contiguous chunks, one per
//            warp.  A lane owns 8 nodes of a 256-node window and keeps the four phase rows of M0 and of
//            M1 at those nodes in REGISTERS (64 values, row r in slot r mod 4); moving to the next
//            observation only reloads the rows that changed.  Per observation a lane reads its 8 node
//            weights (two LDS.128) and issues 72 FFMA; four observations share one transposed warp
//            reduction.
// and an epilogue per unit in fp64 (zero point, coalesced stores, chi^2 in a fixed order).  The
// gradient variant (GRAD) adds CL-weighted node weights (d/dc), M1-only and phase-derivative row sums
// (d/dx1, d/dt0) and d chi^2/d theta.  HBM sees only the per-observation records (the next group's are
// prefetched into L2); the model window is read from L2/L1 about once per (warp, stage).
// Requirements (checked by the host, otherwise sb_hoist.cuh / sb_kernels.cuh run): fp32, uniform band
// grids, n_phase in [4, 4096], n_cl <= NCL, n_bands <= 64.
#pragma once
#include "sb_internal.h"
#include "sb_kernels.cuh"
#include "sb_hoist.cuh"

namespace sbt {

using sbh::HColour;
using sbh::HSeg;
using sbh::HUnitTmp;
using sbh::kMaxSeg;

constexpr int kWarps = 16;
constexpr int kThreads = kWarps * 32;
constexpr int kSlots = 32;        // items (unit, band) per stage
constexpr int kW = 512;           // node weights per item slot (one window segment)
constexpr int kPassSeg = kW / 32; // phase-A passes per window segment
constexpr int kNPL = 8;           // nodes per lane in phase B
constexpr int kWinB = 32 * kNPL;  // nodes per phase-B window
constexpr int kBins = 2048;       // bins of the (band, phase row) counting sort
constexpr int kMaxBands = 64;

// One item (segment, band) of the current stage.
struct TItem {
    int32_t n_in;    // in-range band samples (0: nothing to do)
    int32_t ncell;   // model cells spanned
    int32_t g_first; // first cell
    int32_t wbase;   // index of the first in-range sample in the staged weight table
    int32_t cmode;
    int32_t n_lo;    // first node that carries a weight (g_first - 1, >= -1)
    int32_t n_end;   // one past the last node that carries a weight (g_last + 3)
    float c0, ha_hi, ha_lo, inv_ha, hal, r_first, lin_a, lin_b;
};

struct TSmem {
    size_t w, at, res, ws, info, key, hist, bstart, segs, utmp, items, win, x1, misc, total;
    // grad: two weight sets per item (value, d/dc) in the same At array (half as many item slots), two
    // float4 of phase weights (value, d/dt0) and four results per observation
    __host__ __device__ TSmem(int n_band_total, int cap, bool grad, int n_items)
    {
        size_t o = 0;
        at = o; o += (size_t)kSlots * kW * sizeof(float);
        ws = o; o += (size_t)cap * sizeof(float4) * (grad ? 2 : 1);
        w = o; o += (size_t)((n_band_total + 3) & ~3) * sizeof(float);
        res = o; o += (size_t)cap * sizeof(float) * (grad ? 4 : 1);
        info = o; o += (size_t)cap * sizeof(uint32_t);
        hist = o; o += (size_t)kBins * sizeof(int32_t);
        bstart = o; o += (size_t)(kMaxBands + 4) * sizeof(int32_t);
        key = o; o += (size_t)((cap + 7) & ~7) * sizeof(uint16_t);
        o = (o + 15) & ~(size_t)15;
        segs = o; o += (size_t)kMaxSeg * sizeof(HSeg);
        utmp = o; o += (size_t)kMaxSeg * sizeof(HUnitTmp);
        items = o; o += (size_t)n_items * sizeof(TItem);          // every (band, segment) of a round
        win = o; o += (size_t)2 * kMaxBands * sizeof(int32_t);     // [lo | end][band]: union node window
        x1 = o; o += (size_t)kSlots * sizeof(float);              // [item slot of a stage]
        misc = o; o += 64;
        total = o;
    }
};

__device__ __forceinline__ float4 lds128(const float *p) { return *reinterpret_cast<const float4 *>(p); }

// ---- geometry of one item (segment S, band b): one thread.  Same decisions as sbh::run_item: the
// in-range sample range [j_lo, j_hi) in fp64 (reading G9), the window of model cells, the colour mode.
// unscaled = true (gradient kernel): lin_a / lin_b describe CL itself, not CL times c log2(e).
__device__ __forceinline__ void item_geometry(const SbHParams &P, const HSeg &S, int b, TItem &I, bool unscaled)
{
    const SbModelParams &mp = P.mp;
    const int nW = mp.n_wave;
    I.n_in = 0;
    I.n_lo = 0;
    I.n_end = 0;
    const int boff = __ldg(P.band_off + b);
    const int nb = __ldg(P.band_off + b + 1) - boff;
    const double lam_first = __ldg(P.band_lam_first + b);
    const double h = __ldg(P.band_h + b);
    const double opz = S.opz, inv_opz = S.inv_opz;
    const double dl_lo = mp.l0 * opz - lam_first;
    const double dl_hi = (mp.l0 + (double)(nW - 1) * mp.dl) * opz - lam_first;
    const double *__restrict__ dlam = P.band_dlam + boff;
    int j_lo = (int)fmin(fmax(ceil(dl_lo / h), 0.0), (double)nb);
    while (j_lo > 0 && __ldg(dlam + j_lo - 1) >= dl_lo) --j_lo;
    while (j_lo < nb && __ldg(dlam + j_lo) < dl_lo) ++j_lo;
    int j_hi = (int)fmin(fmax(floor(dl_hi / h) + 1.0, 0.0), (double)nb);
    while (j_hi < nb && __ldg(dlam + j_hi) <= dl_hi) ++j_hi;
    while (j_hi > 0 && __ldg(dlam + j_hi - 1) > dl_hi) --j_hi;
    if (j_lo >= j_hi) return; // band entirely outside the model grid: results stay 0 (G3)

    const double a_d = inv_opz / mp.dl;                      // cells per observer-frame Angstrom
    const double ub = (lam_first * inv_opz - mp.l0) / mp.dl; // u of dlam = 0
    const double ha = h * a_d;                               // cells per band sample
    const double u_lo = (double)j_lo * ha + ub;
    const double u_hi = (double)(j_hi - 1) * ha + ub;
    const int g_first = min(max((int)floor(u_lo), 0), nW - 2);
    const int g_last = min(max((int)floor(u_hi), 0), nW - 2);
    I.n_in = j_hi - j_lo;
    I.g_first = g_first;
    I.ncell = g_last - g_first + 1;
    I.wbase = boff + j_lo;
    I.c0 = (float)(u_lo - (double)g_first);
    I.ha_hi = (float)ha;
    I.ha_lo = (float)(ha - (double)I.ha_hi);
    I.inv_ha = (float)(1.0 / ha);
    const double al_d = inv_opz * mp.cl_inv_span;
    const double be_d = (lam_first * inv_opz - mp.cl_b) * mp.cl_inv_span;
    const double hal = h * al_d;
    const double r_a = (double)j_lo * hal + be_d, r_b = (double)(j_hi - 1) * hal + be_d;
    I.hal = (float)hal;
    I.r_first = (float)r_a;
    I.lin_a = 0.f;
    I.lin_b = 0.f;
    const double r_min = fmin(r_a, r_b), r_max = fmax(r_a, r_b);
    const double margin = 1e-4;
    int cmode = sb::CM_GENERIC;
    if (r_min >= mp.r_lo + margin && r_max <= mp.r_hi - margin) {
        cmode = sb::CM_INSIDE;
    } else if (r_min >= mp.r_hi + margin) { // arg = p_hi + s_hi (r - r_hi)
        cmode = sb::CM_LINEAR;
        const double sl = unscaled ? mp.s_hi : (double)S.s_hi, pv = unscaled ? mp.p_hi : (double)S.p_hi;
        I.lin_b = (float)sl;
        I.lin_a = (float)(pv - sl * mp.r_hi);
    } else if (r_max <= mp.r_lo - margin) {
        cmode = sb::CM_LINEAR;
        const double sl = unscaled ? mp.s_lo : (double)S.s_lo, pv = unscaled ? mp.p_lo : (double)S.p_lo;
        I.lin_b = (float)sl;
        I.lin_a = (float)(pv - sl * mp.r_lo);
    }
    I.cmode = cmode;
    I.n_lo = g_first - 1; // nodes g_first-1 .. g_last+2 carry weights
    I.n_end = g_last + 3;
}

// ---- phase A: node weights of one item -> At slot (one warp) --------------------------------------
// All items of a band use the BAND's node grid: node w_lo + 32 q + l belongs to lane l of pass q, and
// the slot holds passes [q_lo, q_hi) of it (one window segment).  Lane l also owns CELL node + 1.
// Node n takes w_{-1} of cell n+1 (this lane), w_0 of cell n (lane - 1), w_1 of cell n-1 (lane - 2)
// and w_2 of cell n-2 (lane - 3); lanes 0..2 take them from the previous pass (carried in registers;
// when the segment starts inside the item's window the pass before it is recomputed for its carries).
// Passes outside the item's own nodes [n_lo, n_end) are zero filled.
// The loop walks TWO passes (cells gq and gq + 32 of the lane) per iteration: the two cells' colour-law /
// ex2 / moment chains are independent, which hides their fixed latencies with only four warps per
// scheduler.  GRAD: the colour law is evaluated unscaled (CL itself; exponent = CL * c log2(e)) and a
// second set of moments, weighted by CL, gives the node weights of d/dc (at_slot + kW).
template <int NCL, int CM, bool GRAD>
__device__ __forceinline__ void phase_a_passes(const SbModelParams &mp, const HSeg &S, const TItem &I, int w_lo,
                                               int q_start, int q_a, int q_b, int q_lo,
                                               const float *__restrict__ s_w, float *__restrict__ at_slot, int lane)
{
    constexpr unsigned FULL = 0xffffffffu;
    HColour<NCL> col;
#pragma unroll
    for (int q = 0; q < NCL; ++q) col.a[q] = GRAD ? (float)mp.cl[q] : S.cl[q];
    col.r_lo = (float)mp.r_lo;
    col.r_hi = (float)mp.r_hi;
    col.s_lo = GRAD ? (float)mp.s_lo : S.s_lo;
    col.s_hi = GRAD ? (float)mp.s_hi : S.s_hi;
    col.lin_a = I.lin_a;
    col.lin_b = I.lin_b;
    const float cs = (float)(S.cc * 1.4426950408889634); // GRAD: exponent in log2 units = CL * cs
    const int nW = mp.n_wave;
    const float c0 = I.c0, inv_ha = I.inv_ha, ha_hi = I.ha_hi, ha_lo = I.ha_lo, hal = I.hal, r_first = I.r_first;
    const int n_in = I.n_in, ncell = I.ncell;
    auto jstart = [&](int x) { // first band sample (relative to the first in-range one) of cell x
        int j = (int)ceilf(((float)x - c0) * inv_ha);
        j = min(max(j, 0), n_in); // x <= 0 gives j <= 0 because c0 >= 0
        if (x >= ncell) j = n_in;
        return j;
    };
    float pa0 = 0.f, pa1 = 0.f, pa2 = 0.f;
    float pc0 = 0.f, pc1 = 0.f, pc2 = 0.f; // GRAD: carries of the d/dc weights
    int gq = w_lo + 32 * q_start + lane + 1 - I.g_first; // this lane's cell (first pass) relative to g_first
    int carry = jstart(gq);                                // lane 0: start of its cell
    const float *wbase = s_w + I.wbase;
    float *outp = at_slot + (q_start - q_lo) * 32 + lane;
    auto from_left = [&](float cur, float prev, int d) {
        const float a = __shfl_up_sync(FULL, cur, d);
        const float b = __shfl_sync(FULL, prev, (lane - d) & 31);
        return lane >= d ? a : b;
    };
    // moments of the lane's two cells (.x: cell g, .y: cell g + 32) -> weights on their four nodes (Keys
    // a = -1/2; linear in border cells, G2), packed; the lane's node of each pass takes its cell's w_-1
    // and w_0, w_1, w_2 of the three cells to the left (previous pass for lanes 0..2: p0..p2, which for
    // the second cell are the first cell's values)
    auto node_weights = [&](int g, float2 m0, float2 m1, float2 m2, float2 m3, float &p0, float &p1, float &p2) {
        const float2 half = make_float2(0.5f, 0.5f);
        float2 am = __fmul2_rn(half, __fadd2_rn(__ffma2_rn(make_float2(2.0f, 2.0f), m2, make_float2(-m3.x, -m3.y)),
                                                 make_float2(-m1.x, -m1.y)));
        float2 a0 = __ffma2_rn(make_float2(1.5f, 1.5f), m3, __ffma2_rn(make_float2(-2.5f, -2.5f), m2, m0));
        float2 a1 = __fmul2_rn(half, __ffma2_rn(make_float2(-3.0f, -3.0f), m3, __ffma2_rn(make_float2(4.0f, 4.0f), m2, m1)));
        float2 a2 = __fmul2_rn(half, __fadd2_rn(m3, make_float2(-m2.x, -m2.y)));
        if (g <= 0 || g >= nW - 2) {
            am.x = 0.f; a0.x = m0.x - m1.x; a1.x = m1.x; a2.x = 0.f;
        }
        if (g + 32 <= 0 || g + 32 >= nW - 2) {
            am.y = 0.f; a0.y = m0.y - m1.y; a1.y = m1.y; a2.y = 0.f;
        }
        const float2 l0 = make_float2(from_left(a0.x, p0, 1), from_left(a0.y, a0.x, 1));
        const float2 l1 = make_float2(from_left(a1.x, p1, 2), from_left(a1.y, a1.x, 2));
        const float2 l2 = make_float2(from_left(a2.x, p2, 3), from_left(a2.y, a2.x, 3));
        p0 = a0.y;
        p1 = a1.y;
        p2 = a2.y;
        return __fadd2_rn(__fadd2_rn(__fadd2_rn(am, l0), l1), l2);
    };
#pragma unroll 1
    for (int q = q_start; q < q_b; q += 2) {
        const int jeA = jstart(gq + 1), jeB = jstart(gq + 33);
        int jsA = __shfl_up_sync(FULL, jeA, 1), jsB = __shfl_up_sync(FULL, jeB, 1);
        const int lastA = __shfl_sync(FULL, jeA, 31);
        if (lane == 0) { jsA = carry; jsB = lastA; }
        carry = __shfl_sync(FULL, jeB, 31);
        const int cntA = jeA - jsA, cntB = jeB - jsB;
        const float fA = (float)jsA, fB = (float)jsB;
        const float2 f2 = make_float2(fA, fB);
        const float *wpA = wbase + jsA, *wpB = wbase + jsB;
        const int km = __reduce_max_sync(FULL, max(cntA, cntB));
        // moments of the two cells as packed FP32 pairs (.x: cell gq, .y: cell gq + 32): FFMA2 / FMUL2 /
        // FADD2 take one issue slot per pair and give each element the scalar sequence of operations
        float2 m0 = make_float2(0.f, 0.f), m1 = m0, m2 = m0, m3 = m0;
        float2 n0 = m0, n1 = m0, n2 = m0, n3 = m0; // GRAD: weighted by CL
        const float2 hh = make_float2(ha_hi, ha_hi), ll = make_float2(hal, hal), cc2 = make_float2(cs, cs);
        // u_js - cell, and the reduced wavelength of the first sample, of both cells
        float2 t2v = __fadd2_rn(__ffma2_rn(f2, make_float2(ha_lo, ha_lo),
                                           __ffma2_rn(f2, hh, make_float2(-(float)gq, -(float)(gq + 32)))),
                                make_float2(c0, c0));
        float2 r2v = __ffma2_rn(f2, ll, make_float2(r_first, r_first));
#pragma unroll 1
        for (int k = 0; k < km; ++k) { // one sample of each of the two cells per trip
            float2 w = make_float2(0.f, 0.f);
            if (k < cntA) w.x = wpA[k];
            if (k < cntB) w.y = wpB[k];
            const float2 cl = col.template arg2<CM>(r2v);
            const float2 ar = GRAD ? __fmul2_rn(cl, cc2) : cl;
            const float2 e = __fmul2_rn(make_float2(sb::exp_scaled(ar.x), sb::exp_scaled(ar.y)), w);
            const float2 tt = __fmul2_rn(t2v, t2v);
            const float2 ttt = __fmul2_rn(tt, t2v);
            m0 = __fadd2_rn(m0, e);
            m1 = __ffma2_rn(e, t2v, m1);
            m2 = __ffma2_rn(e, tt, m2);
            m3 = __ffma2_rn(e, ttt, m3);
            if (GRAD) {
                const float2 g = __fmul2_rn(e, cl);
                n0 = __fadd2_rn(n0, g);
                n1 = __ffma2_rn(g, t2v, n1);
                n2 = __ffma2_rn(g, tt, n2);
                n3 = __ffma2_rn(g, ttt, n3);
            }
            t2v = __fadd2_rn(t2v, hh);
            r2v = __fadd2_rn(r2v, ll);
        }
        const bool stA = q >= q_a, stB = q + 1 >= q_a && q + 1 < q_b;
        const float2 at = node_weights(I.g_first + gq, m0, m1, m2, m3, pa0, pa1, pa2);
        if (stA) outp[0] = at.x;
        if (stB) outp[32] = at.y;
        if (GRAD) {
            const float2 ac = node_weights(I.g_first + gq, n0, n1, n2, n3, pc0, pc1, pc2);
            if (stA) outp[kW] = ac.x;
            if (stB) outp[kW + 32] = ac.y;
        }
        outp += 64;
        gq += 64;
    }
}

template <int NCL, bool GRAD>
__device__ __forceinline__ void phase_a_item(const SbModelParams &mp, const HSeg &S, const TItem &I, int w_lo,
                                             int q_lo, int q_hi, const float *__restrict__ s_w,
                                             float *__restrict__ at_slot, int lane)
{
    // passes of the band grid that hold nodes of this item
    int q_a = q_hi, q_b = q_hi, qa = 0;
    if (I.n_in > 0) {
        qa = (I.n_lo - w_lo) >> 5;
        const int qb = (I.n_end - 1 - w_lo) >> 5;
        q_a = min(max(qa, q_lo), q_hi);
        q_b = max(min(qb + 1, q_hi), q_a);
    }
    // zero fill up to a whole 128-node half window: phase B reads the slot in halves
    const int q_fill = q_lo + (((q_hi - q_lo) + 3) & ~3);
    for (int q = q_lo; q < q_a; ++q) {
        at_slot[(q - q_lo) * 32 + lane] = 0.f;
        if (GRAD) at_slot[kW + (q - q_lo) * 32 + lane] = 0.f;
    }
    for (int q = q_b; q < q_fill; ++q) {
        at_slot[(q - q_lo) * 32 + lane] = 0.f;
        if (GRAD) at_slot[kW + (q - q_lo) * 32 + lane] = 0.f;
    }
    if (q_a >= q_b) return;
    const int q_start = q_a > qa ? q_a - 1 : q_a;
    if (I.cmode == sb::CM_INSIDE)
        phase_a_passes<NCL, sb::CM_INSIDE, GRAD>(mp, S, I, w_lo, q_start, q_a, q_b, q_lo, s_w, at_slot, lane);
    else if (I.cmode == sb::CM_LINEAR)
        phase_a_passes<NCL, sb::CM_LINEAR, GRAD>(mp, S, I, w_lo, q_start, q_a, q_b, q_lo, s_w, at_slot, lane);
    else
        phase_a_passes<NCL, sb::CM_GENERIC, GRAD>(mp, S, I, w_lo, q_start, q_a, q_b, q_lo, s_w, at_slot, lane);
}

// ---- phase B: observations [i_lo, i_hi) of the sorted list (all of one band) on one warp ----------
// Node window of 256 (TWO = true) or 128 nodes starting at node n0, whose weights start at float
// a_off of every item slot: lane l owns nodes n0 + 4 l .. + 3 and n0 + 128 + 4 l .. + 3.
// All products of the contraction are issued as packed FP32 pairs (FFMA2 / FMUL2, sm_100): the kernel is
// bound by instruction issue, not by the FMA pipe, and a pair takes one issue slot.  A pair is two
// neighbouring nodes of the lane; each element sees exactly the scalar sequence of fused multiply-adds.
struct RowRegs {
    float2 m0[4][kNPL / 2], m1[4][kNPL / 2]; // [slot = row mod 4][node pair]
};

template <bool TWO>
__device__ __forceinline__ void load_row(RowRegs &R, int s, const float *__restrict__ p0, const float *__restrict__ p1,
                                         bool ok_lo, bool ok_hi)
{
    float4 a = make_float4(0.f, 0.f, 0.f, 0.f), b = a, c = a, d = a;
    if (ok_lo) {
        a = __ldg(reinterpret_cast<const float4 *>(p0));
        c = __ldg(reinterpret_cast<const float4 *>(p1));
    }
    if (TWO && ok_hi) {
        b = __ldg(reinterpret_cast<const float4 *>(p0 + 128));
        d = __ldg(reinterpret_cast<const float4 *>(p1 + 128));
    }
    R.m0[s][0] = make_float2(a.x, a.y); R.m0[s][1] = make_float2(a.z, a.w);
    R.m1[s][0] = make_float2(c.x, c.y); R.m1[s][1] = make_float2(c.z, c.w);
    if (TWO) {
        R.m0[s][2] = make_float2(b.x, b.y); R.m0[s][3] = make_float2(b.z, b.w);
        R.m1[s][2] = make_float2(d.x, d.y); R.m1[s][3] = make_float2(d.z, d.w);
    }
}

template <bool TWO>
__device__ __forceinline__ void phase_b_window(const SbHParams &P, int n0, const float *__restrict__ s_at_l,
                                               const float *__restrict__ s_x1, const float4 *__restrict__ s_ws,
                                               const uint32_t *__restrict__ s_info, float *__restrict__ res, int i_lo,
                                               int i_hi, int lane)
{
    const int ld = P.mp.ld;
    RowRegs R;
    int held[4] = {-1, -1, -1, -1};
    int rb_held = -1;
    const int col = n0 + SB_PAD_L + 4 * lane; // column of this lane's first node (multiple of 4)
    const bool ok_lo = col >= 0 && col + 4 <= ld;
    const bool ok_hi = col + 128 >= 0 && col + 132 <= ld;
    const float *p0 = P.m0 + col, *p1 = P.m1 + col;
#pragma unroll
    for (int s = 0; s < 4; ++s)
#pragma unroll
        for (int q = 0; q < kNPL / 2; ++q) { R.m0[s][q] = make_float2(0.f, 0.f); R.m1[s][q] = make_float2(0.f, 0.f); }

    auto rows = [&](int rb) { // rows rb .. rb+3, row r in register slot r mod 4: reload only what changed
        if (rb == rb_held) return;
        rb_held = rb;
#pragma unroll
        for (int s = 0; s < 4; ++s) {
            const int row = rb + ((s - rb) & 3);
            if (held[s] != row) {
                const ptrdiff_t ro = (ptrdiff_t)row * ld;
                load_row<TWO>(R, s, p0 + ro, p1 + ro, ok_lo, ok_hi);
                held[s] = row;
            }
        }
    };
    // NOBS observations that use the same four rows (already in R) at once: 4 NOBS independent chains of
    // packed pairs per 128-node half.  x1 is applied to M1 first (t = M0 + x1 M1), so an observation
    // keeps only its four row weights and x1 in registers.
    auto compute = [&](auto nobs_tag, int i, float *out) {
        constexpr int NOBS = decltype(nobs_tag)::value;
        float2 ws[NOBS][4], xx[NOBS], a2[NOBS];
        const float *ap[NOBS];
#pragma unroll
        for (int o = 0; o < NOBS; ++o) {
            const int slot = (int)(s_info[i + o] & 31u);
            const float4 w4 = s_ws[i + o];
            const float x1 = s_x1[slot];
            xx[o] = make_float2(x1, x1);
            ws[o][0] = make_float2(w4.x, w4.x); ws[o][1] = make_float2(w4.y, w4.y);
            ws[o][2] = make_float2(w4.z, w4.z); ws[o][3] = make_float2(w4.w, w4.w);
            ap[o] = s_at_l + slot * kW;
            a2[o] = make_float2(0.f, 0.f); // even / odd nodes of the lane
        }
#pragma unroll
        for (int hf = 0; hf < (TWO ? 2 : 1); ++hf) {
            float2 av[NOBS][2];
#pragma unroll
            for (int o = 0; o < NOBS; ++o) {
                const float4 t = lds128(ap[o] + 128 * hf);
                av[o][0] = make_float2(t.x, t.y);
                av[o][1] = make_float2(t.z, t.w);
            }
#pragma unroll
            for (int q = 0; q < 2; ++q) {
#pragma unroll
                for (int o = 0; o < NOBS; ++o) {
                    float2 r = __fmul2_rn(ws[o][0], __ffma2_rn(xx[o], R.m1[0][2 * hf + q], R.m0[0][2 * hf + q]));
#pragma unroll
                    for (int s = 1; s < 4; ++s)
                        r = __ffma2_rn(ws[o][s], __ffma2_rn(xx[o], R.m1[s][2 * hf + q], R.m0[s][2 * hf + q]), r);
                    a2[o] = __ffma2_rn(av[o][q], r, a2[o]);
                }
            }
        }
#pragma unroll
        for (int o = 0; o < NOBS; ++o) out[o] = a2[o].x + a2[o].y;
    };
    auto rb_of = [&](int i) { return (int)((s_info[i] >> 5) & 4095u); };
    auto pair_of = [&](int i, float *out) { // observations i and i + 1
        const int rbA = rb_of(i), rbB = rb_of(i + 1);
        rows(rbA);
        if (rbA == rbB) {
            compute(std::integral_constant<int, 2>{}, i, out);
        } else {
            compute(std::integral_constant<int, 1>{}, i, out);
            rows(rbB);
            compute(std::integral_constant<int, 1>{}, i + 1, out + 1);
        }
    };
    auto one = [&](int i) -> float {
        float v;
        rows(rb_of(i));
        compute(std::integral_constant<int, 1>{}, i, &v);
        return v;
    };

    int i = i_lo;
    for (; i + 4 <= i_hi; i += 4) {
        float acc[4];
        pair_of(i, acc);
        pair_of(i + 2, acc + 2);
        const float v = sbh::warp_reduce_transpose<4>(acc, lane); // lane L: total of observation i + (L >> 3)
        if ((lane & 7) == 0) res[s_info[i + (lane >> 3)] >> 17] += v;
    }
    if (i < i_hi) {
        float acc[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
        for (int j = 0; j < 3; ++j)
            if (i + j < i_hi) acc[j] = one(i + j);
        const float v = sbh::warp_reduce_transpose<4>(acc, lane);
        if ((lane & 7) == 0 && i + (lane >> 3) < i_hi) res[s_info[i + (lane >> 3)] >> 17] += v;
    }
    __syncwarp();
}

// Gradient variant of phase B: 128-node window (4 nodes per lane), four sums per observation --
// value, M1-only (d/dx1), CL-weighted node weights (d/dc), phase-derivative weights (d/dt0; the factor
// -1/((1+z) dP) is folded into the weights) -- PAPER.md:45, 49; BASELINE.json north_star (a8).
__device__ __forceinline__ void phase_b_window_grad(const SbHParams &P, int n0, const float *__restrict__ s_at_l,
                                                    const float *__restrict__ s_x1, const float4 *__restrict__ s_ws,
                                                    const float4 *__restrict__ s_wd,
                                                    const uint32_t *__restrict__ s_info, float *__restrict__ res,
                                                    int cap, int i_lo, int i_hi, int lane)
{
    const int ld = P.mp.ld;
    float2 m0[4][2], m1[4][2]; // [slot = row mod 4][node pair]: packed FP32 pairs as in phase_b_window
    int held[4] = {-1, -1, -1, -1};
    int rb_held = -1;
    const int col = n0 + SB_PAD_L + 4 * lane;
    const bool ok = col >= 0 && col + 4 <= ld;
    const float *p0 = P.m0 + col, *p1 = P.m1 + col;
#pragma unroll
    for (int s = 0; s < 4; ++s)
#pragma unroll
        for (int q = 0; q < 2; ++q) { m0[s][q] = make_float2(0.f, 0.f); m1[s][q] = make_float2(0.f, 0.f); }

    auto one = [&](int i, float *acc) { // acc[0..3] = value, M1-only, d/dc, d/dt0 shares of observation i
        const uint32_t info = s_info[i];
        const int slot = (int)(info & 31u), rb = (int)((info >> 5) & 4095u);
        if (rb != rb_held) {
            rb_held = rb;
#pragma unroll
            for (int s = 0; s < 4; ++s) {
                const int row = rb + ((s - rb) & 3);
                if (held[s] != row) {
                    const ptrdiff_t ro = (ptrdiff_t)row * ld;
                    float4 a = make_float4(0.f, 0.f, 0.f, 0.f), c = a;
                    if (ok) {
                        a = __ldg(reinterpret_cast<const float4 *>(p0 + ro));
                        c = __ldg(reinterpret_cast<const float4 *>(p1 + ro));
                    }
                    m0[s][0] = make_float2(a.x, a.y); m0[s][1] = make_float2(a.z, a.w);
                    m1[s][0] = make_float2(c.x, c.y); m1[s][1] = make_float2(c.z, c.w);
                    held[s] = row;
                }
            }
        }
        const float4 w4 = s_ws[i], d4 = s_wd[i];
        const float x1 = s_x1[slot];
        const float2 xx = make_float2(x1, x1);
        const float2 ws[4] = {make_float2(w4.x, w4.x), make_float2(w4.y, w4.y), make_float2(w4.z, w4.z),
                              make_float2(w4.w, w4.w)};
        const float2 wd[4] = {make_float2(d4.x, d4.x), make_float2(d4.y, d4.y), make_float2(d4.z, d4.z),
                              make_float2(d4.w, d4.w)};
        const float2 vd[4] = {__fmul2_rn(wd[0], xx), __fmul2_rn(wd[1], xx), __fmul2_rn(wd[2], xx), __fmul2_rn(wd[3], xx)};
        const float *ap = s_at_l + slot * (2 * kW);
        const float4 t = lds128(ap), tc = lds128(ap + kW);
        const float2 av[2] = {make_float2(t.x, t.y), make_float2(t.z, t.w)};
        const float2 ac[2] = {make_float2(tc.x, tc.y), make_float2(tc.z, tc.w)};
        float2 s_a = make_float2(0.f, 0.f), s_1 = s_a, s_c = s_a, s_d = s_a; // even / odd nodes
#pragma unroll
        for (int q = 0; q < 2; ++q) {
            float2 r0 = __fmul2_rn(ws[0], m0[0][q]), r1 = __fmul2_rn(ws[0], m1[0][q]), rd = __fmul2_rn(wd[0], m0[0][q]);
#pragma unroll
            for (int s = 1; s < 4; ++s) {
                r0 = __ffma2_rn(ws[s], m0[s][q], r0);
                r1 = __ffma2_rn(ws[s], m1[s][q], r1);
                rd = __ffma2_rn(wd[s], m0[s][q], rd);
            }
#pragma unroll
            for (int s = 0; s < 4; ++s) rd = __ffma2_rn(vd[s], m1[s][q], rd);
            const float2 r = __ffma2_rn(xx, r1, r0);
            s_a = __ffma2_rn(av[q], r, s_a);
            s_1 = __ffma2_rn(av[q], r1, s_1);
            s_c = __ffma2_rn(ac[q], r, s_c);
            s_d = __ffma2_rn(av[q], rd, s_d);
        }
        const float a = s_a.x + s_a.y, a1 = s_1.x + s_1.y, a_c = s_c.x + s_c.y, a_d = s_d.x + s_d.y;
        acc[0] = a; acc[1] = a1; acc[2] = a_c; acc[3] = a_d;
    };

    for (int i = i_lo; i < i_hi; i += 4) {
        float acc[16];
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            if (i + j < i_hi) one(i + j, acc + 4 * j);
            else { acc[4 * j] = 0.f; acc[4 * j + 1] = 0.f; acc[4 * j + 2] = 0.f; acc[4 * j + 3] = 0.f; }
        }
        // lane L ends with value (L >> 1) = 4 * observation + component
        const float v = sbh::warp_reduce_transpose<16>(acc, lane);
        const int vi = lane >> 1, j = vi >> 2, comp = vi & 3;
        if ((lane & 1) == 0 && i + j < i_hi) res[comp * cap + (int)(s_info[i + j] >> 17)] += v;
    }
    __syncwarp();
}

// Phase of observation o of segment S: first loaded phase row rb (rows rb .. rb+3) and the weights of
// those rows (Keys a = -1/2, linear in the border cells -- readings G1, G2), scalar work in fp64.
// Returns false when the phase is outside the grid (zero flux, reading G3).
__device__ __forceinline__ bool obs_phase(const SbModelParams &mp, const HSeg &S, float t, int &rb, double (&wrow)[4],
                                          double (&drow)[4])
{
    const int nP = mp.n_phase;
    const double p = ((double)t - S.t0) * S.inv_opz;
    const double up = (p - mp.p0) * mp.inv_dp;
    if (!((up >= 0.0) && (up <= (double)(nP - 1)))) return false;
    const int kp = min((int)floor(up), nP - 2);
    double wv[4], wd[4];
    // d/dt0 of the weights: d tau/d t0 = -1/((1+z) dP)
    sb::phase_weights(up - (double)kp, (kp == 0) || (kp == nP - 2), -S.inv_opz * mp.inv_dp, wv, wd);
    rb = min(max(kp - 1, 0), nP - 4);
    const int shift = (kp - 1) - rb; // row rb + k carries Keys weight index k - shift
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const int src = k - shift;
        double w = 0.0, d = 0.0;
        if (src == 0) { w = wv[0]; d = wd[0]; }
        if (src == 1) { w = wv[1]; d = wd[1]; }
        if (src == 2) { w = wv[2]; d = wd[2]; }
        if (src == 3) { w = wv[3]; d = wd[3]; }
        wrow[k] = w;
        drow[k] = d;
    }
    return true;
}

// ---- the kernel ---------------------------------------------------------------------------------
// GRAD = true: also d m/d(x0, x1, c, t0) and d chi^2/d theta (row a8); half as many item slots (two
// weight sets per item), 128-node windows in phase B.
template <int NCL, bool GRAD>
__global__ void __launch_bounds__(kThreads, 1) sb_tiled_kernel(const __grid_constant__ SbHParams P)
{
    constexpr int NSL = GRAD ? kSlots / 2 : kSlots; // item slots per stage
    constexpr int ATS = GRAD ? 2 * kW : kW;         // floats per item slot
    extern __shared__ __align__(16) unsigned char smem_raw[];
    constexpr unsigned FULL = 0xffffffffu;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const SbModelParams &mp = P.mp;
    const TSmem L(P.n_band_total, P.cap, GRAD, P.n_bands * P.group_units);
    float *s_at = reinterpret_cast<float *>(smem_raw + L.at);
    float4 *s_ws = reinterpret_cast<float4 *>(smem_raw + L.ws);
    float *s_w = reinterpret_cast<float *>(smem_raw + L.w);
    float *res = reinterpret_cast<float *>(smem_raw + L.res);
    uint32_t *s_info = reinterpret_cast<uint32_t *>(smem_raw + L.info);
    uint16_t *s_key = reinterpret_cast<uint16_t *>(smem_raw + L.key);
    int *hist = reinterpret_cast<int *>(smem_raw + L.hist);
    int *bstart = reinterpret_cast<int *>(smem_raw + L.bstart);
    HSeg *segs = reinterpret_cast<HSeg *>(smem_raw + L.segs);
    HUnitTmp *utmp = reinterpret_cast<HUnitTmp *>(smem_raw + L.utmp);
    TItem *items_all = reinterpret_cast<TItem *>(smem_raw + L.items);   // [band][segment]
    int *win_all = reinterpret_cast<int *>(smem_raw + L.win);           // [lo: kMaxBands | end: kMaxBands]
    float *x1_all = reinterpret_cast<float *>(smem_raw + L.x1);         // [kSlots]
    int *misc = reinterpret_cast<int *>(smem_raw + L.misc);             // [0] group, [1] n_seg, [2] n_ev, [3] next unit, [4] next offset
    double *carry = reinterpret_cast<double *>(smem_raw + L.misc + 24); // chi^2 [, d chi^2] of a unit split over rounds
    const float4 *s_wd = s_ws + P.cap;                                  // GRAD: d/dt0 phase weights

    for (int i = tid; i < P.n_band_total; i += kThreads) s_w[i] = __ldg(P.band_w + i);
    const long long n_units = (long long)P.n_sn * P.n_samples;
    const int G = P.group_units, CAP = P.cap;
    const long long n_groups = (n_units + G - 1) / G;
    const bool want_chi = P.out_chi2 != nullptr || (GRAD && P.out_dchi2 != nullptr);
    const int nP = mp.n_phase, n_bands = P.n_bands;
    const int nq = max(1, min(nP - 3, kBins / n_bands)); // phase-row bins per band
    constexpr uint16_t kNoKey = 0xffffu;

    // Groups are claimed one ahead (misc[5] = the next group of this CTA) so that the records of the
    // next group can be pulled into L2 while the current one is computed.
    if (tid == 0) misc[5] = (int)atomicAdd(P.counter, 1u);
    for (;;) {
        __syncthreads();
        const long long group = (long long)(unsigned)misc[5];
        __syncthreads();
        if (group >= n_groups) break;
        if (tid == kThreads - 1) misc[5] = (int)atomicAdd(P.counter, 1u); // read again after many barriers
        const long long pos0 = group * G;
        const int npos = (int)min((long long)G, n_units - pos0);
        if (tid < npos) { // unit -> supernova (z-ordered), observation range
            const long long pos = pos0 + tid;
            const int si = (int)(pos / P.n_samples);
            const int ks = (int)(pos - (long long)si * P.n_samples);
            const int sn = P.perm ? __ldg(P.perm + si) : si;
            HUnitTmp t;
            t.sn = sn;
            t.unit = sn * P.n_samples + ks;
            t.o_lo = __ldg(P.obs_offset + sn);
            t.n = __ldg(P.obs_offset + sn + 1) - t.o_lo;
            utmp[tid] = t;
        }
        if (tid == 0) { misc[3] = 0; misc[4] = 0; }
        __syncthreads();

        for (;;) {
            const int cur_u = misc[3];
            __syncthreads();
            if (cur_u >= npos) break;
            // ---- round: consecutive units whose observations fit the result array (a unit larger
            // than the array is processed alone, CAP observations at a time)
            if (tid == 0) {
                int u = misc[3], off = misc[4], n_ev = 0, n_seg = 0;
                while (u < npos && n_seg < NSL) {
                    const int rem = utmp[u].n - off;
                    HSeg &S = segs[n_seg];
                    if (rem <= CAP - n_ev) {
                        S.unit = u; S.o_lo = off; S.n = rem; S.e_begin = n_ev; S.first = (off == 0); S.last = 1;
                        n_ev += rem; ++n_seg; ++u; off = 0;
                    } else if (n_ev == 0) {
                        S.unit = u; S.o_lo = off; S.n = CAP; S.e_begin = 0; S.first = (off == 0); S.last = 0;
                        n_ev = CAP; ++n_seg; off += CAP;
                        break;
                    } else {
                        break;
                    }
                }
                misc[1] = n_seg; misc[2] = n_ev; misc[3] = u; misc[4] = off;
            }
            for (int i = tid; i < kBins; i += kThreads) hist[i] = 0;
            if (tid < kMaxBands) { win_all[tid] = 0x7fffffff; win_all[kMaxBands + tid] = -0x7fffffff; }
            __syncthreads();
            const int n_seg = misc[1], n_ev = misc[2];
            if (tid < n_seg) { // segment parameters (S.unit / S.o_lo hold group-local values until here)
                HSeg &S = segs[tid];
                const HUnitTmp t = utmp[S.unit];
                const int off = S.o_lo;
                const int ks = t.unit - t.sn * P.n_samples;
                S.unit = t.unit;
                S.sn = t.sn;
                S.o_lo = t.o_lo + off;
                S.out_base = (long long)t.o_lo * P.n_samples + (long long)ks * t.n + off;
                const double z = (double)__ldg(P.z + t.sn);
                const double cc = (double)__ldg(P.c + t.unit);
                S.opz = 1.0 + z;
                S.inv_opz = 1.0 / S.opz;
                S.x0 = (double)__ldg(P.x0 + t.unit);
                S.x1 = __ldg(P.x1 + t.unit);
                S.t0 = (double)__ldg(P.t0 + t.unit);
                S.cc = cc;
                const double cscale = cc * 1.4426950408889634; // exponent in log2 units (ex2)
#pragma unroll
                for (int q = 0; q < SB_MAX_CL; ++q) S.cl[q] = (float)(mp.cl[q] * cscale);
                S.s_lo = (float)(mp.s_lo * cscale);
                S.s_hi = (float)(mp.s_hi * cscale);
                S.p_lo = (float)(mp.p_lo * cscale);
                S.p_hi = (float)(mp.p_hi * cscale);
            }
            for (int e = tid; e < n_ev; e += kThreads) {
                res[e] = 0.f;
                if (GRAD) { res[CAP + e] = 0.f; res[2 * CAP + e] = 0.f; res[3 * CAP + e] = 0.f; }
            }
            __syncthreads();

            // ---- a1: counting sort of the round's observations by (band, phase row) ----------------
            auto seg_of = [&](int e) {
                int lo = 0, hi = n_seg - 1;
                while (lo < hi) {
                    const int mid = (lo + hi + 1) >> 1;
                    if (segs[mid].e_begin <= e) lo = mid;
                    else hi = mid - 1;
                }
                return lo;
            };
            for (int e = tid; e < n_ev; e += kThreads) {
                const int sg = seg_of(e);
                const HSeg &S = segs[sg];
                const int o = S.o_lo + (e - S.e_begin);
                const int b = __ldg(P.band + o);
                uint16_t key = kNoKey;
                if ((unsigned)b < (unsigned)n_bands) {
                    int rb;
                    double wrow[4], drow[4];
                    if (obs_phase(mp, S, __ldg(P.time + o), rb, wrow, drow)) {
                        key = (uint16_t)(b * nq + (rb * nq) / (nP - 3));
                        atomicAdd(&hist[key], 1);
                    }
                }
                s_key[e] = key;
            }
            __syncthreads();
            if (tid < 32) { // exclusive scan of the bins, start of every band's run
                constexpr int PER = kBins / 32;
                int s = 0;
                for (int k = 0; k < PER; ++k) s += hist[tid * PER + k];
                int incl = s;
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) {
                    const int v = __shfl_up_sync(FULL, incl, o);
                    if (tid >= o) incl += v;
                }
                int run = incl - s;
                for (int k = 0; k < PER; ++k) {
                    const int c = hist[tid * PER + k];
                    hist[tid * PER + k] = run;
                    run += c;
                }
                if (tid == 31) bstart[n_bands] = run;
                __syncwarp();
                for (int b = tid; b < n_bands; b += 32) bstart[b] = hist[b * nq];
            }
            __syncthreads();
            const int bps = max(1, NSL / n_seg); // bands per stage
            for (int e = tid; e < n_ev; e += kThreads) {
                const uint16_t key = s_key[e];
                if (key == kNoKey) continue;
                const int sg = seg_of(e);
                const HSeg &S = segs[sg];
                const int o = S.o_lo + (e - S.e_begin);
                int rb = 0;
                double wrow[4] = {0.0, 0.0, 0.0, 0.0}, drow[4] = {0.0, 0.0, 0.0, 0.0};
                obs_phase(mp, S, __ldg(P.time + o), rb, wrow, drow);
                float wsl[4], wdl[4]; // register slot s holds the row congruent to s mod 4
#pragma unroll
                for (int s = 0; s < 4; ++s) {
                    const int k = (s - rb) & 3;
                    wsl[s] = (float)(k == 0 ? wrow[0] : k == 1 ? wrow[1] : k == 2 ? wrow[2] : wrow[3]);
                    wdl[s] = (float)(k == 0 ? drow[0] : k == 1 ? drow[1] : k == 2 ? drow[2] : drow[3]);
                }
                const int b = (int)key / nq;
                const int slot = (b % bps) * n_seg + sg; // item slot inside the band's stage
                const int pos = atomicAdd(&hist[key], 1);
                s_ws[pos] = make_float4(wsl[0], wsl[1], wsl[2], wsl[3]);
                if (GRAD) s_ws[CAP + pos] = make_float4(wdl[0], wdl[1], wdl[2], wdl[3]);
                s_info[pos] = (uint32_t)slot | ((uint32_t)rb << 5) | ((uint32_t)e << 17);
            }

            // ---- geometry of every item (band, segment) of the round, union node window of every band:
            // all threads at once, so the latency of its dependent loads is paid once per round
            for (int it = tid; it < n_bands * n_seg; it += kThreads) {
                const int b = it / n_seg, sg = it - b * n_seg;
                TItem &I = items_all[it];
                I.n_in = 0; I.n_lo = 0; I.n_end = 0;
                if (bstart[b + 1] > bstart[b] && segs[sg].n > 0) item_geometry(P, segs[sg], b, I, GRAD);
                if (I.n_in > 0) {
                    atomicMin(&win_all[b], I.n_lo & ~3); // multiple of 4: 16-byte aligned row loads
                    atomicMax(&win_all[kMaxBands + b], I.n_end);
                }
            }
            if (tid < NSL) x1_all[tid] = segs[tid % n_seg].x1; // item slot -> x1 of its segment
            __syncthreads(); // sorted records, items and band windows are visible

            // ---- L2 prefetch of the next group's records (one lane per unit, last warp, first round)
            if (warp == kWarps - 1 && cur_u == 0) {
                const long long pos = (long long)(unsigned)misc[5] * G + lane;
                if (lane < G && (long long)(unsigned)misc[5] < n_groups && pos < n_units) {
                    const int si = (int)(pos / P.n_samples);
                    const int sn = P.perm ? __ldg(P.perm + si) : si;
                    const int o_lo = __ldg(P.obs_offset + sn), n = __ldg(P.obs_offset + sn + 1) - o_lo;
                    auto pf = [](const void *p) { asm volatile("prefetch.global.L2 [%0];" ::"l"(p)); };
                    const long long unit = (long long)sn * P.n_samples + (pos - (long long)si * P.n_samples);
                    pf(P.z + sn); pf(P.x0 + unit); pf(P.x1 + unit); pf(P.c + unit); pf(P.t0 + unit);
                    for (int o = 0; o < n + 31; o += 32) { // one 128-byte line of every array per step
                        const int oo = o_lo + min(o, n - 1);
                        if (n <= 0) break;
                        pf(P.time + oo);
                        pf(P.band + oo);
                        if (P.zp) pf(P.zp + oo);
                        if (P.flux) { pf(P.flux + oo); pf(P.fluxerr + oo); }
                    }
                }
            }

            // ---- stages: as many whole bands as fit the item slots; two CTA barriers per stage and
            // window segment
            const int n_stage = (n_bands + bps - 1) / bps;
            for (int st = 0; st < n_stage; ++st) {
                const int b0 = st * bps, nbs = min(bps, n_bands - b0), n_items = nbs * n_seg;
                const TItem *items = items_all + b0 * n_seg;
                const int *win_lo = win_all + b0, *win_end = win_all + kMaxBands + b0;
                const float *s_x1 = x1_all;
                int n_wseg = 0; // window segments of kW nodes: the widest band of the stage decides
                for (int bl = 0; bl < nbs; ++bl) {
                    const int len = win_end[bl] - win_lo[bl];
                    if (len > 0) n_wseg = max(n_wseg, (len + kW - 1) / kW);
                }
                for (int wseg = 0; wseg < n_wseg; ++wseg) {
                    // phase A: node weights of every item on its band's node grid
                    for (int it = warp; it < n_items; it += kWarps) {
                        const int bl = it / n_seg, sg = it - bl * n_seg;
                        const int w_lo = win_lo[bl], len = win_end[bl] - w_lo;
                        if (len <= 0) continue;
                        const int np_b = (len + 31) >> 5;
                        const int q_lo = wseg * kPassSeg, q_hi = min(q_lo + kPassSeg, np_b);
                        if (q_lo >= q_hi) continue;
                        phase_a_item<NCL, GRAD>(mp, segs[sg], items[it], w_lo, q_lo, q_hi, s_w, s_at + (size_t)it * ATS, lane);
                    }
                    __syncthreads();
                    // phase B: contraction with the model rows, observations in (band, phase row) order
                    for (int bl = 0; bl < nbs; ++bl) {
                        const int w_lo = win_lo[bl], len = win_end[bl] - w_lo;
                        if (len <= 0) continue;
                        const int np_w = min(kPassSeg, ((len + 31) >> 5) - wseg * kPassSeg);
                        if (np_w <= 0) continue;
                        const int lo = bstart[b0 + bl], n = bstart[b0 + bl + 1] - lo;
                        const int per = (((n + kWarps - 1) / kWarps) + 3) & ~3;
                        const int i_lo = lo + warp * per, i_hi = min(i_lo + per, lo + n);
                        if (i_lo >= i_hi) continue;
                        const int n_half = (np_w * 32 + 127) >> 7; // 128-node halves of this segment
                        if constexpr (GRAD) {
                            for (int h0 = 0; h0 < n_half; ++h0)
                                phase_b_window_grad(P, w_lo + wseg * kW + 128 * h0, s_at + 128 * h0 + 4 * lane, s_x1, s_ws,
                                                    s_wd, s_info, res, CAP, i_lo, i_hi, lane);
                        } else {
                            for (int h0 = 0; h0 < n_half; h0 += 2) {
                                const int n0 = w_lo + wseg * kW + 128 * h0;
                                const float *at_l = s_at + 128 * h0 + 4 * lane;
                                if (h0 + 1 < n_half) phase_b_window<true>(P, n0, at_l, s_x1, s_ws, s_info, res, i_lo, i_hi, lane);
                                else phase_b_window<false>(P, n0, at_l, s_x1, s_ws, s_info, res, i_lo, i_hi, lane);
                            }
                        }
                    }
                    __syncthreads();
                }
            }

            // ---- epilogue: one warp per segment; a6 zero point (fp64), flux [, gradient] out (coalesced),
            // a7 chi^2 [, a8 d chi^2/d theta = -2 sum (f - m)/sigma^2 dm/dtheta] in a fixed order
            float zp_last = __int_as_float(0x7fc00000); // NaN: never equal
            double zp_pow = 1.0;
            for (int sg = warp; sg < n_seg; sg += kWarps) {
                const HSeg &S = segs[sg];
                constexpr int NS = GRAD ? 5 : 1;
                double sum[NS];
#pragma unroll
                for (int k = 0; k < NS; ++k) sum[k] = 0.0;
                for (int i = lane; i < S.n; i += 32) {
                    const int o = S.o_lo + i;
                    const int b = __ldg(P.band + o);
                    const double qnan = __longlong_as_double(0x7ff8000000000000LL);
                    double m = qnan, dm[4] = {qnan, qnan, qnan, qnan};
                    if ((unsigned)b < (unsigned)P.n_bands) {
                        double sc = 1.0;
                        if (P.zp != nullptr) { // 10^(0.4 zp): recomputed only when zp changes (usually never)
                            const float zpv = __ldg(P.zp + o);
                            if (zpv != zp_last) {
                                zp_last = zpv;
                                zp_pow = exp10(0.4 * (double)zpv);
                            }
                            sc = zp_pow * __ldg(P.band_zpab_inv + b);
                        }
                        const double raw = (double)res[S.e_begin + i];
                        m = sc * S.x0 * raw;
                        if (GRAD) {
                            dm[0] = sc * raw;
                            dm[1] = sc * S.x0 * (double)res[CAP + S.e_begin + i];
                            dm[2] = sc * S.x0 * (double)res[2 * CAP + S.e_begin + i];
                            dm[3] = sc * S.x0 * (double)res[3 * CAP + S.e_begin + i];
                        }
                    }
                    if (P.out_flux) P.out_flux[S.out_base + i] = (float)m;
                    if (GRAD && P.out_dflux)
                        reinterpret_cast<float4 *>(P.out_dflux)[S.out_base + i] =
                            make_float4((float)dm[0], (float)dm[1], (float)dm[2], (float)dm[3]);
                    if (want_chi) {
                        const double f = (double)__ldg(P.flux + o), e = (double)__ldg(P.fluxerr + o);
                        const double qv = (f - m) / e;
                        sum[0] += qv * qv;
                        if (GRAD) {
                            const double g = -2.0 * (f - m) / (e * e);
#pragma unroll
                            for (int k = 0; k < 4; ++k) sum[1 + k] += g * dm[k];
                        }
                    }
                }
                if (want_chi) {
#pragma unroll
                    for (int k = 0; k < NS; ++k) sum[k] = sb::warp_sum(sum[k]);
                    if (lane == 0) {
                        double total[NS];
#pragma unroll
                        for (int k = 0; k < NS; ++k) total[k] = (S.first ? 0.0 : carry[k]) + sum[k];
                        if (S.last) {
                            if (P.out_chi2) P.out_chi2[S.unit] = (float)total[0];
                            if (GRAD && P.out_dchi2)
                                reinterpret_cast<float4 *>(P.out_dchi2)[S.unit] =
                                    make_float4((float)total[1], (float)total[2], (float)total[3], (float)total[4]);
                        } else {
#pragma unroll
                            for (int k = 0; k < NS; ++k) carry[k] = total[k];
                        }
                    }
                }
            }
            __syncthreads();
        }
    }
}

} // namespace sbt
