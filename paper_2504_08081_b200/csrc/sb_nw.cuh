// sb_nw.cuh -- the pipelined node-weight kernel (sm_100a), fp32, forward and gradient.
//
// Same sums per evaluation as sb_kernels.cuh, with the band integral
// re-associated into NODE WEIGHTS (an exact exchange of two finite sums):
//     raw_o = sum_s ws_s(o) * D_s(o),   D_s(o) = sum_l At[l] * (M0 + x1 M1)[rb_o + s][l],
//     At[l] = sum_j ew_j w_{l-i_j}(tau_j),   ew_j = exp(c CL(lambda_j/(1+z))) W_j
// (w = Keys a = -1/2 weights, reading G1; ws = the four phase-row weights of the
// observation).  At depends on (unit, band) only -- an ITEM -- and is shared by all
// observations of the item.
//
// Work decomposition.  The units (supernova x sample) are taken in redshift order (sb_zorder_* kernels of sb_hoist.cuh) and cut
// into GROUPS of z-neighbours; CTA c of a persistent grid owns groups c, c + gridDim, ... (static: no
// counter, no per-call mutable state).  A group is processed in ROUNDS of at most `cap` observations and
// `NSL` units.  Per round:
//   prologue  every observation: phase -> first model row rb and the four row weights (fp64 scalar work,
//             once), counting sort by (band, rb) in shared memory (parallel scan); every item: geometry
//             (from the pack, or computed here) and the union node window of every band.
//   stages    a STAGE is a set of bands x one 256-node window segment.  Two phases per stage:
//     phase A  one warp per item: lanes own model cells, walk the band samples of their cells (colour
//              factor x folded weight -> moments sum ew tau^p), turn the moments into node weights and
//              store At[item][0..256) in shared memory;
//     phase B  the stage's observations, sorted by rb, are cut into one contiguous chunk per warp; a lane
//              keeps the four phase rows of M0 and M1 at its (up to 8) nodes in REGISTERS and slides that
//              row window as rb grows; per observation it reads its node weights (LDS.128) and
//              accumulates D_s with packed FP32 pairs (FFMA2: 8 per node pair), applies the row weights to
//              the four partial sums and joins a transposed warp reduction of four observations.
//   The node-weight array is DOUBLE BUFFERED: in one super-step every warp runs phase A of stage s+1 and
//   phase B of stage s (half of the warps in the opposite order, so that both kinds of work are in
//   flight on every scheduler) and there is ONE CTA barrier per stage.
//   epilogue  per unit in fp64: zero point, coalesced stores, chi^2 (and d chi^2) in a fixed order.
// The gradient variant (GRAD) adds CL-weighted node weights (d/dc), the M1-only sums (d/dx1) and the
// phase-derivative row weights (d/dt0).
// Band grids need not be uniform (tabulated filters): the NU variant of the kernel reads, beside
// the folded weight W_j of a band sample, its offset delta_j = lambda_j - (lambda_first + j h) from the band's
// mean-step grid, so that the position inside the model cell and the colour-law argument are those of the true
// wavelength; which samples belong to a model cell is found by a local search from the uniform-grid guess.
// Requirements (checked by the host, otherwise sb_kernels.cuh runs): fp32, n_phase in [4, 4096], n_cl <= NCL,
// n_bands <= 64.
#pragma once
#include "sb_internal.h"
#include "sb_kernels.cuh"
#include "sb_hoist.cuh"

// Checked build (python -m paper_2504_08081_b200.build --checked, -DSB_CHECKED): every shared-memory index
// computed below is compared with the bound of its array and the kernel traps on a violation (the next
// CUDA call then fails: SB_ECUDA).  Stands in for compute-sanitizer, which this GPU pool does not allow
// (profiles/r2_sanitizer.md).  Compiles to nothing in the product build.
#ifdef SB_CHECKED
#define SB_CHECK(cond) do { if (!(cond)) __trap(); } while (0)
#else
#define SB_CHECK(cond) do { } while (0)
#endif

namespace sbn {

using sbh::HColour;

constexpr int kSlotW = 256;           // node weights per item slot (one window segment)
constexpr int kPassSeg = kSlotW / 32; // phase-A passes per window segment
constexpr int kMaxBands = 64;

// CTA shape.  NW = 16: one CTA of 16 warps per SM; NW = 8: two CTAs of 8 warps per SM (half the shared
// memory each), so that the barriers, prologue and epilogue of one CTA overlap the other's stages.  The
// work per warp (items per stage, observations per chunk) is the same in both.
template <int NW> struct Cfg {
    static constexpr int kWarps = NW;
    static constexpr int kThreads = NW * 32;
    static constexpr int kSlots = 2 * NW;                  // item slots per buffer (forward); gradient: half
    static constexpr int kBins = NW == 16 ? 2048 : 1024;   // bins of the (band, phase row) counting sort
    static constexpr int kMaxSeg = kSlots;                 // segments (units) per round
    static constexpr int kCapFwd = NW == 16 ? 3072 : 1280; // observations per round
    static constexpr int kCapGrad = NW == 16 ? 1536 : 640;
};

// Geometry of one item (supernova, band): depends on z and the band only (never on theta), so the pack
// (sb_pack_observations, saltband.cu) can hold it.  64 bytes, loaded as four 16-byte words.
struct __align__(16) NItem {
    int32_t n_in;    // in-range band samples (0: nothing to do)
    int32_t ncell;   // model cells spanned
    int32_t g_first; // first cell
    int32_t wbase;   // index of the first in-range sample in the staged weight table
    int32_t cmode;   // colour-law mode of the whole item (sb::CM_*)
    int32_t n_lo;    // first node that carries a weight (g_first - 1, >= -1)
    int32_t n_end;   // one past the last node that carries a weight (g_last + 3)
    int32_t pad_;
    float c0, ha_hi, ha_lo, inv_ha; // u of the first sample ON THE MEAN-STEP GRID minus g_first; cells per (mean) band step (split), inverse
    float hal, r_first;             // reduced-wavelength step per (mean) band step, value at the first sample of the mean-step grid
    float lin_a, lin_b;             // CM_LINEAR: CL = lin_a + lin_b r (unscaled)
};
static_assert(sizeof(NItem) == 64, "NItem is loaded as four float4");

// One segment = a contiguous run of observations of one unit (a whole unit unless it exceeds the round).
struct __align__(16) NSeg {
    double x0, t0, opz, inv_opz, cc;
    long long out_base;  // out_flux index of the segment's first observation
    int32_t unit, sn, o_lo, n, e_begin, first, last;
    float x1;
    float cl[SB_MAX_CL]; // forward: colour-law coefficients times c log2(e)
    float s_lo, s_hi;    // continuation slopes, same scaling
    float cs;            // c log2(e)
    int32_t pad_;
};

struct NUnit {           // per unit of the group (all rounds)
    int32_t unit, sn, o_lo, n;
    float z, x0, x1, c, t0;
};

struct NSmem {
    size_t at, ws, res, info, w, hist, wsum, bstart, segs, units, items, win, x1, slot_tab, misc, carry, total;
    __host__ __device__ NSmem(int n_band_total, int cap, bool grad, int n_items, int nw, bool nu)
    {
        const int kSlots = 2 * nw, kWarps = nw, kMaxSeg = 2 * nw, kBins = nw == 16 ? 2048 : 1024;
        size_t o = 0;
        at = o; o += (size_t)2 * kSlots * kSlotW * sizeof(float);
        ws = o; o += (size_t)cap * sizeof(float4) * (grad ? 2 : 1);
        res = o; o += (size_t)cap * sizeof(float) * (grad ? 4 : 1);
        info = o; o += (size_t)cap * sizeof(uint32_t);
        w = o; o += (size_t)((n_band_total + 3) & ~3) * (nu ? sizeof(float2) : sizeof(float)); // W_j or {W_j, delta_j}
        hist = o; o += (size_t)kBins * sizeof(int32_t);
        wsum = o; o += (size_t)kWarps * sizeof(int32_t);
        bstart = o; o += (size_t)(kMaxBands + 4) * sizeof(int32_t);
        o = (o + 15) & ~(size_t)15;
        segs = o; o += (size_t)kMaxSeg * sizeof(NSeg);
        units = o; o += (size_t)kMaxSeg * sizeof(NUnit);
        o = (o + 15) & ~(size_t)15;
        items = o; o += (size_t)n_items * sizeof(NItem);          // every (band, segment) of a round
        win = o; o += (size_t)2 * kMaxBands * sizeof(int32_t);     // [lo | end][band]: union node window
        x1 = o; o += (size_t)kSlots * sizeof(float2);             // [item slot] {x1, x1}
        slot_tab = o; o += (size_t)kSlots * sizeof(int32_t);       // [item slot] band-in-stage | segment << 8
        misc = o; o += 64;
        o = (o + 15) & ~(size_t)15;
        carry = o; o += 8 * sizeof(double);                        // chi^2 [, d chi^2] of a unit split over rounds
        total = o;
    }
};

// Kernel parameter block.
struct SbNParams {
    SbModelParams mp;
    const float *mx;                  // M0 [n_phase][mp.ld]; M1 the same SBN_M1_OFF bytes further (sb_internal.h)
    int32_t n_bands, n_band_total;
    const int32_t *band_off;
    const double *band_lam_first, *band_zpab_inv, *band_h, *band_dlam;
    const float *band_w;              // [n_band_total] folded weights W_j
    const float2 *band_wd;            // [n_band_total] {W_j, delta_j} (NU kernels)
    int32_t n_sn, n_samples;
    const int32_t *obs_offset;
    const float *time, *zp, *z, *x0, *x1, *c, *t0;
    const int32_t *band;
    const float *flux, *fluxerr;      // may be NULL
    float *out_flux, *out_chi2;       // may be NULL
    float *out_dflux, *out_dchi2;     // gradient kernel only; may be NULL
    const int32_t *perm;              // z-ordered supernova indices (pack or workspace), or NULL
    const NItem *geom;                // [n_sn][n_bands] item geometry of the pack, or NULL (computed here)
    const int32_t *live, *n_live;     // fit driver: [n_units] 0 = skip the unit; [1] 0 = nothing to do (or NULL)
    int32_t n_groups;                 // groups: unit range of group i = [i n_units / n_groups, (i+1) n_units / n_groups)
    int32_t cap;                      // observations per round
};

// Shared-memory accesses of the hot loops go through 32-bit shared-state-space addresses (one cvta at
// kernel start) instead of generic pointers: no 64-bit address arithmetic and no per-access window-base
// computation (S2UR + ULEA, each a scoreboard stall).  An array is accessed either only through these
// or only through C++ pointers between two CTA barriers.
__device__ __forceinline__ uint32_t smem_addr(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ float4 lds128(uint32_t a)
{
    float4 v;
    asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(a));
    return v;
}
__device__ __forceinline__ float2 lds64(uint32_t a)
{
    float2 v;
    asm volatile("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(v.x), "=f"(v.y) : "r"(a));
    return v;
}
__device__ __forceinline__ float lds32(uint32_t a)
{
    float v;
    asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(a));
    return v;
}
__device__ __forceinline__ uint32_t lds32u(uint32_t a)
{
    uint32_t v;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(a));
    return v;
}
__device__ __forceinline__ void sts32(uint32_t a, float v) { asm volatile("st.shared.f32 [%0], %1;" ::"r"(a), "f"(v)); }

// Read-only global loads at a compile-time byte offset from a pointer.  TAG (the register slot the row goes
// to) is spelled into the instruction text so that the loads of different switch cases are different
// instructions for the compiler: it then writes each case's rows straight into that case's registers
// instead of merging the cases into one load followed by predicated register moves.
template <int TAG, int OFF> __device__ __forceinline__ float4 ldg128_at(const float *p)
{
    float4 v;
    asm volatile("{\n\t// row slot %5\n\tld.global.nc.v4.f32 {%0, %1, %2, %3}, [%4+%6];\n\t}"
                 : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "l"(p), "n"(TAG), "n"(OFF));
    return v;
}
template <int TAG, int OFF> __device__ __forceinline__ float2 ldg64_at(const float *p)
{
    float2 v;
    asm volatile("{\n\t// row slot %3\n\tld.global.nc.v2.f32 {%0, %1}, [%2+%4];\n\t}"
                 : "=f"(v.x), "=f"(v.y) : "l"(p), "n"(TAG), "n"(OFF));
    return v;
}

struct NShared { // shared-state-space addresses of the arrays phase B reads
    uint32_t info, ws, wd, x1, res;
    int32_t cap;
    int32_t n_slots; // item slots per node-weight buffer (checked build)
};

// Colour-law modes of an item beyond sb::CM_*: the item's samples cross only ONE end of [cl_lo, cl_hi]
// (one clamp and one fixed slope instead of two clamps and a slope select per sample).
enum { CM_CROSS_HI = 3, CM_CROSS_LO = 4 };

// Exponent argument of the colour factor for two wavelengths at once (packed FP32 pairs).
template <int NCL, int CM> __device__ __forceinline__ float2 colour_arg2(const HColour<NCL> &col, float2 r)
{
    if constexpr (CM == CM_CROSS_HI || CM == CM_CROSS_LO) {
        constexpr bool HI = CM == CM_CROSS_HI;
        const float lim = HI ? col.r_hi : col.r_lo, sl = HI ? col.s_hi : col.s_lo;
        const float2 rc = HI ? make_float2(fminf(r.x, lim), fminf(r.y, lim)) : make_float2(fmaxf(r.x, lim), fmaxf(r.y, lim));
        const float2 d = __fadd2_rn(r, make_float2(-rc.x, -rc.y));
        float2 p = make_float2(col.a[NCL - 1], col.a[NCL - 1]);
#pragma unroll
        for (int q = NCL - 2; q >= 0; --q) p = __ffma2_rn(p, rc, make_float2(col.a[q], col.a[q]));
        return __ffma2_rn(make_float2(sl, sl), d, p);
    } else {
        return col.template arg2<CM>(r);
    }
}

// ---- geometry of one item (redshift z, band b): one thread.  The in-range sample range [j_lo, j_hi) is
// decided in fp64 (reading G9), then the window of model cells and the colour-law mode.
struct NBandsView {
    int32_t n_bands, all_uniform;
    const int32_t *band_off;
    const double *band_lam_first, *band_h, *band_dlam;
};

__device__ __forceinline__ void item_geometry(const SbModelParams &mp, const NBandsView &B, double opz, int b, NItem &I)
{
    const int nW = mp.n_wave;
    I.n_in = 0; I.ncell = 0; I.g_first = 0; I.wbase = 0; I.cmode = sb::CM_GENERIC; I.n_lo = 0; I.n_end = 0; I.pad_ = 0;
    I.c0 = 0.f; I.ha_hi = 0.f; I.ha_lo = 0.f; I.inv_ha = 0.f; I.hal = 0.f; I.r_first = 0.f; I.lin_a = 0.f; I.lin_b = 0.f;
    const double inv_opz = 1.0 / opz;
    const int boff = __ldg(B.band_off + b);
    const int nb = __ldg(B.band_off + b + 1) - boff;
    const double lam_first = __ldg(B.band_lam_first + b);
    const double h = __ldg(B.band_h + b);
    const double dl_lo = mp.l0 * opz - lam_first;
    const double dl_hi = (mp.l0 + (double)(nW - 1) * mp.dl) * opz - lam_first;
    const double *__restrict__ dlam = B.band_dlam + boff;
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
    // first and last in-range sample at their true wavelengths (the mean-step grid differs on non-uniform grids)
    const double u_lo = __ldg(dlam + j_lo) * a_d + ub;
    const double u_hi = __ldg(dlam + j_hi - 1) * a_d + ub;
    const int g_first = min(max((int)floor(u_lo), 0), nW - 2);
    const int g_last = min(max((int)floor(u_hi), 0), nW - 2);
    I.n_in = j_hi - j_lo;
    I.g_first = g_first;
    I.ncell = g_last - g_first + 1;
    I.wbase = boff + j_lo;
    I.c0 = (float)((double)j_lo * ha + ub - (double)g_first);
    if (B.all_uniform) I.c0 = fmaxf(I.c0, 0.f); // uniform grid: the mean-step grid IS the grid (up to rounding of the table)
    I.ha_hi = (float)ha;
    I.ha_lo = (float)(ha - (double)I.ha_hi);
    I.inv_ha = (float)(1.0 / ha);
    const double al_d = inv_opz * mp.cl_inv_span;
    const double be_d = (lam_first * inv_opz - mp.cl_b) * mp.cl_inv_span;
    const double hal = h * al_d;
    const double r_a = __ldg(dlam + j_lo) * al_d + be_d, r_b = __ldg(dlam + j_hi - 1) * al_d + be_d;
    I.hal = (float)hal;
    I.r_first = (float)((double)j_lo * hal + be_d);
    const double r_min = fmin(r_a, r_b), r_max = fmax(r_a, r_b);
    const double margin = 1e-4;
    int cmode = sb::CM_GENERIC;
    if (r_min >= mp.r_lo + margin) cmode = CM_CROSS_HI; // never below the range: only the upper continuation
    if (r_max <= mp.r_hi - margin) cmode = CM_CROSS_LO; // never above the range
    if (r_min >= mp.r_lo + margin && r_max <= mp.r_hi - margin) {
        cmode = sb::CM_INSIDE;
    } else if (r_min >= mp.r_hi + margin) { // CL = p_hi + s_hi (r - r_hi)
        cmode = sb::CM_LINEAR;
        I.lin_b = (float)mp.s_hi;
        I.lin_a = (float)(mp.p_hi - mp.s_hi * mp.r_hi);
    } else if (r_max <= mp.r_lo - margin) {
        cmode = sb::CM_LINEAR;
        I.lin_b = (float)mp.s_lo;
        I.lin_a = (float)(mp.p_lo - mp.s_lo * mp.r_lo);
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
// The loop walks TWO passes (cells gq and gq + 32 of the lane) per iteration as packed FP32 pairs.
// GRAD: the colour law is evaluated unscaled (CL itself; exponent = CL * c log2(e)) and a second set of
// moments, weighted by CL, gives the node weights of d/dc (at_slot + kSlotW).
template <int NCL, int CM, bool GRAD, bool NU>
__device__ __forceinline__ void phase_a_passes(const SbModelParams &mp, const NSeg &S, const NItem &I, int w_lo,
                                               int q_start, int q_a, int q_b, int q_lo, uint32_t a_w,
                                               uint32_t at_slot, int lane)
{
    constexpr unsigned FULL = 0xffffffffu;
    const float cs = S.cs; // c log2(e)
    HColour<NCL> col;
#pragma unroll
    for (int q = 0; q < NCL; ++q) col.a[q] = GRAD ? (float)mp.cl[q] : S.cl[q];
    col.r_lo = (float)mp.r_lo;
    col.r_hi = (float)mp.r_hi;
    col.s_lo = GRAD ? (float)mp.s_lo : S.s_lo;
    col.s_hi = GRAD ? (float)mp.s_hi : S.s_hi;
    col.lin_a = GRAD ? I.lin_a : I.lin_a * cs;
    col.lin_b = GRAD ? I.lin_b : I.lin_b * cs;
    const int nW = mp.n_wave;
    const float c0 = I.c0, inv_ha = I.inv_ha, ha_hi = I.ha_hi, ha_lo = I.ha_lo, hal = I.hal, r_first = I.r_first;
    const int n_in = I.n_in, ncell = I.ncell;
    const float nc0 = -c0 * inv_ha;
    constexpr uint32_t WS = NU ? 8u : 4u; // bytes per entry of the staged band table: W_j or {W_j, delta_j}
    const uint32_t wbase = a_w + (uint32_t)I.wbase * WS;
    // NU: cells and reduced wavelength per Angstrom (observer frame) of this unit
    const float acell = NU ? (float)(S.inv_opz / mp.dl) : 0.f, alr = NU ? (float)(S.inv_opz * mp.cl_inv_span) : 0.f;
    auto jstart = [&](int x) { // first band sample (relative to the first in-range one) of cell x
        int j = (int)ceilf(__fmaf_rn((float)x, inv_ha, nc0));
        j = min(max(j, 0), n_in); // uniform grids: x <= 0 gives j <= 0 because c0 >= 0
        if (x >= ncell) j = n_in;
        if constexpr (NU) { // local search from the mean-step guess: u_k = c0 + k ha + delta_k acell against x
            if (x <= 0) j = 0;
            if (x > 0 && x < ncell) {
                const float xf = (float)x - c0;
                auto uk = [&](int k) {
                    const float kf = (float)k;
                    return __fmaf_rn(kf, ha_hi, __fmaf_rn(kf, ha_lo, lds64(wbase + (uint32_t)k * 8u).y * acell));
                };
                // the guess's two neighbours are tested at once (independent loads); the loops only run on
                // grids further than one sample from their mean-step grid
                const float below = j > 0 ? uk(j - 1) : -3.0e38f, at = j < n_in ? uk(j) : 3.0e38f;
                if (below >= xf) {
                    --j;
                    while (j > 0 && uk(j - 1) >= xf) --j;
                } else if (at < xf) {
                    ++j;
                    while (j < n_in && uk(j) < xf) ++j;
                }
            }
        }
        return j;
    };
    float pa0 = 0.f, pa1 = 0.f, pa2 = 0.f;
    float pc0 = 0.f, pc1 = 0.f, pc2 = 0.f; // GRAD: carries of the d/dc weights
    int gq = w_lo + 32 * q_start + lane + 1 - I.g_first; // this lane's cell (first pass) relative to g_first
    int carry = jstart(gq);                                // lane 0: start of its cell
    uint32_t outp = at_slot + (uint32_t)((q_start - q_lo) * 32 + lane) * 4u;
    // value of lane - d: of `cur` for lanes >= d, of `prev` (the previous pass) for lanes < d -- one select
    // and one indexed shuffle: the lanes 32 - d .. 31, which nobody reads `cur` from, offer `prev`
    const int src1 = (lane - 1) & 31, src2 = (lane - 2) & 31, src3 = (lane - 3) & 31;
    auto from_left = [&](float cur, float prev, int d, int src) {
        return __shfl_sync(FULL, lane >= 32 - d ? prev : cur, src);
    };
    // moments of the lane's two cells (.x: cell g, .y: cell g + 32) -> weights on their four nodes (Keys
    // a = -1/2; linear in border cells, G2), packed; the lane's node of each pass takes its cell's w_-1
    // and w_0, w_1, w_2 of the three cells to the left
    auto node_weights = [&](int g, bool border, float2 m0, float2 m1, float2 m2, float2 m3, float &p0, float &p1, float &p2) {
        const float2 half = make_float2(0.5f, 0.5f);
        float2 am = __fmul2_rn(half, __fadd2_rn(__ffma2_rn(make_float2(2.0f, 2.0f), m2, make_float2(-m3.x, -m3.y)),
                                                 make_float2(-m1.x, -m1.y)));
        float2 a0 = __ffma2_rn(make_float2(1.5f, 1.5f), m3, __ffma2_rn(make_float2(-2.5f, -2.5f), m2, m0));
        float2 a1 = __fmul2_rn(half, __ffma2_rn(make_float2(-3.0f, -3.0f), m3, __ffma2_rn(make_float2(4.0f, 4.0f), m2, m1)));
        float2 a2 = __fmul2_rn(half, __fadd2_rn(m3, make_float2(-m2.x, -m2.y)));
        if (border) { // some cell of these two passes is a border cell of the model grid (warp uniform, rare)
            if (g <= 0 || g >= nW - 2) {
                am.x = 0.f; a0.x = m0.x - m1.x; a1.x = m1.x; a2.x = 0.f;
            }
            if (g + 32 <= 0 || g + 32 >= nW - 2) {
                am.y = 0.f; a0.y = m0.y - m1.y; a1.y = m1.y; a2.y = 0.f;
            }
        }
        const float2 l0 = make_float2(from_left(a0.x, p0, 1, src1), from_left(a0.y, a0.x, 1, src1));
        const float2 l1 = make_float2(from_left(a1.x, p1, 2, src2), from_left(a1.y, a1.x, 2, src2));
        const float2 l2 = make_float2(from_left(a2.x, p2, 3, src3), from_left(a2.y, a2.x, 3, src3));
        p0 = a0.y;
        p1 = a1.y;
        p2 = a2.y;
        return __fadd2_rn(__fadd2_rn(__fadd2_rn(am, l0), l1), l2);
    };
    const float2 hh = make_float2(ha_hi, ha_hi), ll = make_float2(hal, hal), cc2 = make_float2(cs, cs);
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
        uint32_t wpA = wbase + (uint32_t)jsA * WS, wpB = wbase + (uint32_t)jsB * WS;
        const int km = __reduce_max_sync(FULL, max(cntA, cntB));
        float2 m0 = make_float2(0.f, 0.f), m1 = m0, m2 = m0, m3 = m0;
        float2 n0 = m0, n1 = m0, n2 = m0, n3 = m0; // GRAD: weighted by CL
        // u_js - cell, and the reduced wavelength of the first sample, of both cells
        float2 t2v = __fadd2_rn(__ffma2_rn(f2, make_float2(ha_lo, ha_lo),
                                           __ffma2_rn(f2, hh, make_float2(-(float)gq, -(float)(gq + 32)))),
                                make_float2(c0, c0));
        float2 r2v = __ffma2_rn(f2, ll, make_float2(r_first, r_first));
        auto trip = [&](int k) { // sample k of each of the lane's two cells
            float2 w = make_float2(0.f, 0.f);
            SB_CHECK(k >= cntA || (wpA >= wbase && wpA < wbase + (uint32_t)n_in * WS));
            SB_CHECK(k >= cntB || (wpB >= wbase && wpB < wbase + (uint32_t)n_in * WS));
            float2 tq = t2v, rq = r2v; // position in the cell and reduced wavelength of this sample
            if constexpr (NU) {
                float2 dd = make_float2(0.f, 0.f);
                if (k < cntA) { const float2 v = lds64(wpA); w.x = v.x; dd.x = v.y; }
                if (k < cntB) { const float2 v = lds64(wpB); w.y = v.x; dd.y = v.y; }
                tq = __ffma2_rn(dd, make_float2(acell, acell), t2v);
                rq = __ffma2_rn(dd, make_float2(alr, alr), r2v);
            } else {
                if (k < cntA) w.x = lds32(wpA);
                if (k < cntB) w.y = lds32(wpB);
            }
            wpA += WS;
            wpB += WS;
            const float2 cl = colour_arg2<NCL, CM>(col, rq);
            const float2 ar = GRAD ? __fmul2_rn(cl, cc2) : cl;
            const float2 e = __fmul2_rn(make_float2(sb::exp_scaled(ar.x), sb::exp_scaled(ar.y)), w);
            const float2 tt = __fmul2_rn(tq, tq);
            const float2 ttt = __fmul2_rn(tt, tq);
            m0 = __fadd2_rn(m0, e);
            m1 = __ffma2_rn(e, tq, m1);
            m2 = __ffma2_rn(e, tt, m2);
            m3 = __ffma2_rn(e, ttt, m3);
            if (GRAD) {
                const float2 g = __fmul2_rn(e, cl);
                n0 = __fadd2_rn(n0, g);
                n1 = __ffma2_rn(g, tq, n1);
                n2 = __ffma2_rn(g, tt, n2);
                n3 = __ffma2_rn(g, ttt, n3);
            }
            t2v = __fadd2_rn(t2v, hh);
            r2v = __fadd2_rn(r2v, ll);
        };
        int k = 0;
#pragma unroll 1
        for (; k + 2 <= km; k += 2) { // two trips per iteration: their colour-law / ex2 chains overlap
            trip(k);
            trip(k + 1);
        }
        if (k < km) trip(k);
        const int g = I.g_first + gq, g0 = g - lane; // g0: cell of lane 0 in the first of the two passes
        const bool border = g0 <= 0 || g0 + 63 >= nW - 2;
        const bool stA = q >= q_a, stB = q + 1 >= q_a && q + 1 < q_b;
        const float2 at = node_weights(g, border, m0, m1, m2, m3, pa0, pa1, pa2);
        SB_CHECK(!stA || (outp >= at_slot && outp < at_slot + kSlotW * 4u));
        SB_CHECK(!stB || (outp + 128u >= at_slot && outp + 128u < at_slot + kSlotW * 4u));
        if (stA) sts32(outp, at.x);
        if (stB) sts32(outp + 128u, at.y);
        if (GRAD) {
            const float2 ac = node_weights(g, border, n0, n1, n2, n3, pc0, pc1, pc2);
            if (stA) sts32(outp + kSlotW * 4u, ac.x);
            if (stB) sts32(outp + kSlotW * 4u + 128u, ac.y);
        }
        outp += 256u;
        gq += 64;
    }
}

// One item, window segment passes [q_lo, q_hi) of the band's node grid (q_hi - q_lo <= kPassSeg); the
// slot is zero filled up to a whole 64-node block (phase B reads it in 64-node blocks).
template <int NCL, bool GRAD, bool NU>
__device__ __forceinline__ void phase_a_item(const SbModelParams &mp, const NSeg &S, const NItem &I, int w_lo,
                                             int q_lo, int q_hi, uint32_t a_w, uint32_t at_slot, int lane)
{
    int q_a = q_hi, q_b = q_hi, qa = 0;
    if (I.n_in > 0) {
        qa = (I.n_lo - w_lo) >> 5;
        const int qb = (I.n_end - 1 - w_lo) >> 5;
        q_a = min(max(qa, q_lo), q_hi);
        q_b = max(min(qb + 1, q_hi), q_a);
    }
    // zero fill up to what phase B reads: whole 64-node blocks, and (forward) at least 128 nodes
    const int q_fill = q_lo + ((!GRAD && q_hi - q_lo <= 2) ? 4 : (((q_hi - q_lo) + 1) & ~1));
    SB_CHECK(q_hi - q_lo >= 1 && q_hi - q_lo <= kPassSeg && q_fill - q_lo <= kPassSeg);
    for (int q = q_lo; q < q_a; ++q) {
        sts32(at_slot + (uint32_t)((q - q_lo) * 32 + lane) * 4u, 0.f);
        if (GRAD) sts32(at_slot + (uint32_t)(kSlotW + (q - q_lo) * 32 + lane) * 4u, 0.f);
    }
    for (int q = q_b; q < q_fill; ++q) {
        sts32(at_slot + (uint32_t)((q - q_lo) * 32 + lane) * 4u, 0.f);
        if (GRAD) sts32(at_slot + (uint32_t)(kSlotW + (q - q_lo) * 32 + lane) * 4u, 0.f);
    }
    if (q_a >= q_b) return;
    const int q_start = q_a > qa ? q_a - 1 : q_a;
    if (I.cmode == sb::CM_INSIDE)
        phase_a_passes<NCL, sb::CM_INSIDE, GRAD, NU>(mp, S, I, w_lo, q_start, q_a, q_b, q_lo, a_w, at_slot, lane);
    else if (I.cmode == sb::CM_LINEAR)
        phase_a_passes<NCL, sb::CM_LINEAR, GRAD, NU>(mp, S, I, w_lo, q_start, q_a, q_b, q_lo, a_w, at_slot, lane);
    else if (I.cmode == CM_CROSS_HI)
        phase_a_passes<NCL, CM_CROSS_HI, GRAD, NU>(mp, S, I, w_lo, q_start, q_a, q_b, q_lo, a_w, at_slot, lane);
    else if (I.cmode == CM_CROSS_LO)
        phase_a_passes<NCL, CM_CROSS_LO, GRAD, NU>(mp, S, I, w_lo, q_start, q_a, q_b, q_lo, a_w, at_slot, lane);
    else
        phase_a_passes<NCL, sb::CM_GENERIC, GRAD, NU>(mp, S, I, w_lo, q_start, q_a, q_b, q_lo, a_w, at_slot, lane);
}

// ---- phase B: observations [i_lo, i_hi) of the sorted list (all of one band) on one warp ----------
// Node window starting at node n0 (multiple of 4) whose weights start at float 0 of every item slot:
// N128 blocks of 128 nodes (lane l owns nodes 128 h + 4 l .. + 3: two packed pairs) and, if T64, a tail
// block of 64 nodes (lane l owns nodes 128 N128 + 2 l, + 1: one pair).  Row r of the model lives in
// register slot r mod 4; the observation's row weights are stored pre-rotated to slots.
// Per node pair and row: t = M0 + x1 M1 (FFMA2), D_s += At t (FFMA2); GRAD adds E_s += At M1 (d/dx1) and
// C_s += Atc t (d/dc).  Every element of a pair sees the scalar sequence of fused multiply-adds.
template <int N128, bool T64, bool GRAD>
__device__ __forceinline__ void phase_b_window(const SbNParams &P, int n0, uint32_t a_at, const NShared &SA, bool first,
                                               int i_lo, int i_hi, int lane)
{
    constexpr int NQ = 2 * N128 + (T64 ? 1 : 0); // packed node pairs per lane
    constexpr uint32_t ATS = (GRAD ? 2 * kSlotW : kSlotW) * 4u; // bytes per item slot
    constexpr int NV = GRAD ? 4 : 1;
    float2 M0[4][NQ], M1[4][NQ]; // [slot = row mod 4][node pair]
#pragma unroll
    for (int s = 0; s < 4; ++s)
#pragma unroll
        for (int q = 0; q < NQ; ++q) { M0[s][q] = make_float2(0.f, 0.f); M1[s][q] = make_float2(0.f, 0.f); }
    // the table rows are zero padded on the right by a whole window (saltband.cu: ld), so every load of a
    // window that starts at a node of the grid stays inside its row: no bounds predicates.  One pointer per
    // lane: its nodes of the M0 row of phase row r are at pb + r ld, those of the M1 row SBN_M1_OFF bytes further.
    const float *pb = P.mx + (n0 + SB_PAD_L + 4 * lane);
    const unsigned ld = (unsigned)P.mp.ld;
    const int toff = 128 * N128 - 2 * lane; // tail pair: column n0 + PAD + 128 N128 + 2 lane
    int rb_held = -64; // rows rb_held .. rb_held + 3 are in the registers
    // per-lane shared addresses of the node weights and of the sorted records, made opaque so that they
    // stay in registers (re-materialising them from the thread index costs ~10 instructions per observation)
    uint32_t a_lane = a_at + (uint32_t)lane * 16u, a_rec = SA.info;
    asm volatile("" : "+r"(a_lane), "+r"(a_rec));
    const uint32_t a_tail = a_lane + 512u * N128 - (uint32_t)lane * 8u;
    const uint32_t d_ws = SA.ws - SA.info; // the row weights of record i are at a_rec + d_ws + 16 i

    auto load_slot = [&](auto s_tag, const float *base, int row) {
        constexpr int s = decltype(s_tag)::value;
        const float *pr = base + (size_t)(unsigned)row * ld;
        static_assert(N128 <= 2, "row loads are written out for at most two 128-node blocks");
#pragma unroll
        for (int h = 0; h < N128; ++h) {
            const float4 a = h == 0 ? ldg128_at<s, 0>(pr) : ldg128_at<s, 512>(pr);
            const float4 c = h == 0 ? ldg128_at<s, SBN_M1_OFF>(pr) : ldg128_at<s, SBN_M1_OFF + 512>(pr);
            M0[s][2 * h] = make_float2(a.x, a.y); M0[s][2 * h + 1] = make_float2(a.z, a.w);
            M1[s][2 * h] = make_float2(c.x, c.y); M1[s][2 * h + 1] = make_float2(c.z, c.w);
        }
        if constexpr (T64) {
            M0[s][2 * N128] = ldg64_at<s, 0>(pr + toff);
            M1[s][2 * N128] = ldg64_at<s, SBN_M1_OFF>(pr + toff);
        }
    };
    auto rows = [&](int rb) { // make rows rb .. rb+3 resident; the sorted order makes rb grow slowly
        const int d = rb - rb_held;
        const int first = (d > 0 && d < 4) ? rb_held + 4 : rb; // first row that is not in the registers yet
        rb_held = rb;
        // the lane's pointer, made opaque so that it is formed once per call and not once per slot (the
        // compiler re-materialises it instead of keeping it: 127 live registers)
        const float *base;
        asm volatile("mov.u64 %0, %1;" : "=l"(base) : "l"(pb));
        // one predicated block per register slot (no loop, no switch: the four blocks are straight-line code
        // that writes its own registers): slot s takes the row of [rb, rb + 4) congruent to s mod 4
        { const int row = rb + ((0 - rb) & 3); if (row >= first) load_slot(std::integral_constant<int, 0>{}, base, row); }
        { const int row = rb + ((1 - rb) & 3); if (row >= first) load_slot(std::integral_constant<int, 1>{}, base, row); }
        { const int row = rb + ((2 - rb) & 3); if (row >= first) load_slot(std::integral_constant<int, 2>{}, base, row); }
        { const int row = rb + ((3 - rb) & 3); if (row >= first) load_slot(std::integral_constant<int, 3>{}, base, row); }
    };

    struct Vals { float v[NV]; };
    auto one = [&](int i) { // value [, d/dx1, d/dc, d/dt0] shares of observation i
        Vals out;
        SB_CHECK(i >= 0 && i < SA.cap);
        const uint32_t info = lds32u(a_rec + (uint32_t)i * 4u);
        const uint32_t slot = info & 31u;
        SB_CHECK(slot < (uint32_t)SA.n_slots && (int)(info >> 17) < SA.cap);
        const int rb = (int)((info >> 5) & 4095u);
        if (rb != rb_held) rows(rb);
        const float4 w4 = lds128(a_rec + d_ws + (uint32_t)i * 16u);
        const float2 xx = lds64(SA.x1 + slot * 8u);
        const uint32_t so = slot * ATS;
        float2 at[NQ], ac[GRAD ? NQ : 1];
#pragma unroll
        for (int h = 0; h < N128; ++h) {
            const float4 t = lds128(a_lane + so + 512u * h);
            at[2 * h] = make_float2(t.x, t.y);
            at[2 * h + 1] = make_float2(t.z, t.w);
            if constexpr (GRAD) {
                const float4 u = lds128(a_lane + so + kSlotW * 4u + 512u * h);
                ac[2 * h] = make_float2(u.x, u.y);
                ac[2 * h + 1] = make_float2(u.z, u.w);
            }
        }
        if constexpr (T64) {
            at[2 * N128] = lds64(a_tail + so);
            if constexpr (GRAD) ac[2 * N128] = lds64(a_tail + so + kSlotW * 4u);
        }
        float2 D[4], E[GRAD ? 4 : 1], C[GRAD ? 4 : 1];
#pragma unroll
        for (int s = 0; s < 4; ++s) {
#pragma unroll
            for (int q = 0; q < NQ; ++q) {
                const float2 t = __ffma2_rn(xx, M1[s][q], M0[s][q]);
                if (q == 0) {
                    D[s] = __fmul2_rn(at[0], t);
                    if constexpr (GRAD) {
                        E[s] = __fmul2_rn(at[0], M1[s][0]);
                        C[s] = __fmul2_rn(ac[0], t);
                    }
                } else {
                    D[s] = __ffma2_rn(at[q], t, D[s]);
                    if constexpr (GRAD) {
                        E[s] = __ffma2_rn(at[q], M1[s][q], E[s]);
                        C[s] = __ffma2_rn(ac[q], t, C[s]);
                    }
                }
            }
        }
        const float d0 = D[0].x + D[0].y, d1 = D[1].x + D[1].y, d2 = D[2].x + D[2].y, d3 = D[3].x + D[3].y;
        out.v[0] = __fmaf_rn(w4.w, d3, __fmaf_rn(w4.z, d2, __fmaf_rn(w4.y, d1, w4.x * d0)));
        if constexpr (GRAD) {
            const float4 v4 = lds128(SA.wd + (uint32_t)i * 16u);
            const float e0 = E[0].x + E[0].y, e1 = E[1].x + E[1].y, e2 = E[2].x + E[2].y, e3 = E[3].x + E[3].y;
            const float c0 = C[0].x + C[0].y, c1 = C[1].x + C[1].y, c2 = C[2].x + C[2].y, c3 = C[3].x + C[3].y;
            out.v[1] = __fmaf_rn(w4.w, e3, __fmaf_rn(w4.z, e2, __fmaf_rn(w4.y, e1, w4.x * e0)));
            out.v[2] = __fmaf_rn(w4.w, c3, __fmaf_rn(w4.z, c2, __fmaf_rn(w4.y, c1, w4.x * c0)));
            out.v[3] = __fmaf_rn(v4.w, d3, __fmaf_rn(v4.z, d2, __fmaf_rn(v4.y, d1, v4.x * d0)));
        }
        return out;
    };

    // NOBS observations share one transposed warp reduction (forward: eight, so that the chain of dependent
    // shuffles is paid once per eight; gradient: four, 16 values): NH passes of a four-times unrolled body
    constexpr int NH = GRAD ? 1 : 2, NOBS = 4 * NH;
    for (int i = i_lo; i < i_hi; i += NOBS) {
        float acc[NOBS * NV];
#pragma unroll 1
        for (int half = 0; half < NH; ++half) {
            float q4[4 * NV];
#pragma unroll
            for (int j = 0; j < 4; ++j) { // past the end of the chunk: the last observation again (not stored)
                const Vals r = one(min(i + 4 * half + j, i_hi - 1));
#pragma unroll
                for (int v = 0; v < NV; ++v) q4[NV * j + v] = r.v[v];
            }
#pragma unroll
            for (int k = 0; k < 4 * NV; ++k) {
                if (NH == 1 || half == 0) acc[k] = q4[k];
                else acc[(NH - 1) * 4 * NV + k] = q4[k];
            }
        }
        // lane L ends with value (L >> SH): observation (L >> SH) / NV, component (L >> SH) % NV
        constexpr int SH = GRAD ? 1 : 2;
        const float v = sbh::warp_reduce_transpose<NOBS * NV>(acc, lane);
        const int vi = lane >> SH, j = vi / NV, comp = vi % NV;
        if ((lane & ((1 << SH) - 1)) == 0 && i + j < i_hi) {
            const uint32_t e = lds32u(SA.info + (uint32_t)(i + j) * 4u) >> 17;
            const uint32_t ra = SA.res + (uint32_t)(comp * SA.cap) * 4u + e * 4u;
            sts32(ra, first ? v : v + lds32(ra));
        }
    }
    __syncwarp();
}

// Phase of an observation of segment S: first loaded phase row rb (rows rb .. rb+3) and the weights of
// those rows (Keys a = -1/2, linear in the border cells -- readings G1, G2), scalar work in fp64.
// Returns false when the phase is outside the grid (zero flux, reading G3).
__device__ __forceinline__ bool obs_phase(const SbModelParams &mp, const NSeg &S, float t, int &rb, double (&wrow)[4],
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
template <int NCL, bool GRAD, bool NU>
__global__ void __launch_bounds__(16 * 32, 1) sb_nw_kernel(const __grid_constant__ SbNParams P)
{
    constexpr int NW = 16; // one CTA of 16 warps per SM (two CTAs of 8 warps were measured slower: DESIGN.md section 9)
    constexpr int kWarps = Cfg<NW>::kWarps, kThreads = Cfg<NW>::kThreads, kSlots = Cfg<NW>::kSlots;
    constexpr int kBins = Cfg<NW>::kBins, kCapFwd = Cfg<NW>::kCapFwd, kCapGrad = Cfg<NW>::kCapGrad;
    constexpr int NSL = GRAD ? kSlots / 2 : kSlots;     // item slots per buffer
    constexpr int ATS = GRAD ? 2 * kSlotW : kSlotW;     // floats per item slot
    constexpr int BUF = kSlots * kSlotW;                // floats per buffer
    constexpr int KPT = ((GRAD ? kCapGrad : kCapFwd) + kThreads - 1) / kThreads; // observations per thread in the prologue
    extern __shared__ __align__(16) unsigned char smem_raw[];
    constexpr unsigned FULL = 0xffffffffu;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const SbModelParams &mp = P.mp;
    const int n_bands = P.n_bands, CAP = P.cap;
    const NSmem L(P.n_band_total, CAP, GRAD, n_bands * NSL, NW, NU);
    float *s_at = reinterpret_cast<float *>(smem_raw + L.at);
    float4 *s_ws = reinterpret_cast<float4 *>(smem_raw + L.ws);
    float *s_w = reinterpret_cast<float *>(smem_raw + L.w);
    float *res = reinterpret_cast<float *>(smem_raw + L.res);
    uint32_t *s_info = reinterpret_cast<uint32_t *>(smem_raw + L.info);
    int *hist = reinterpret_cast<int *>(smem_raw + L.hist);
    int *wsum = reinterpret_cast<int *>(smem_raw + L.wsum);
    int *bstart = reinterpret_cast<int *>(smem_raw + L.bstart);
    NSeg *segs = reinterpret_cast<NSeg *>(smem_raw + L.segs);
    NUnit *units = reinterpret_cast<NUnit *>(smem_raw + L.units);
    NItem *items_all = reinterpret_cast<NItem *>(smem_raw + L.items);   // [band][segment]
    int *win_all = reinterpret_cast<int *>(smem_raw + L.win);           // [lo: kMaxBands | end: kMaxBands]
    float2 *s_x1 = reinterpret_cast<float2 *>(smem_raw + L.x1);         // [item slot]
    int *misc = reinterpret_cast<int *>(smem_raw + L.misc);             // [1] n_seg, [2] n_ev, [3] next unit, [4] next offset
    double *carry = reinterpret_cast<double *>(smem_raw + L.carry);
    int *slot_tab = reinterpret_cast<int *>(smem_raw + L.slot_tab);     // [item slot] band-in-stage | segment << 8
    const uint32_t a_at = smem_addr(s_at), a_w = smem_addr(s_w);
    const NShared SA{smem_addr(s_info), smem_addr(s_ws), smem_addr(s_ws + CAP), smem_addr(s_x1), smem_addr(res), CAP, NSL};

    if (P.n_live != nullptr && __ldg(P.n_live) == 0) return; // fit driver: every lane has stopped
    if constexpr (NU) {
        float2 *s_wd = reinterpret_cast<float2 *>(smem_raw + L.w);
        for (int i = tid; i < P.n_band_total; i += kThreads) s_wd[i] = __ldg(P.band_wd + i);
    } else {
        for (int i = tid; i < P.n_band_total; i += kThreads) s_w[i] = __ldg(P.band_w + i);
    }
    const long long n_units = (long long)P.n_sn * P.n_samples;
    const long long n_groups = P.n_groups;
    const bool want_chi = P.out_chi2 != nullptr || (GRAD && P.out_dchi2 != nullptr);
    const int nP = mp.n_phase;
    const int nq = max(1, min(nP - 3, kBins / n_bands)); // phase-row bins per band
    const NBandsView BV{n_bands, NU ? 0 : 1, P.band_off, P.band_lam_first, P.band_h, P.band_dlam};
    auto unit_lo = [&](long long g) { return (g * n_units) / n_groups; };
    auto pf = [](const void *p) { asm volatile("prefetch.global.L2 [%0];" ::"l"(p)); };

    for (long long group = blockIdx.x; group < n_groups; group += gridDim.x) {
        const long long pos0 = unit_lo(group);
        const int npos = (int)(unit_lo(group + 1) - pos0);
        __syncthreads(); // the previous group's epilogue is done with units/segs
        if (tid < npos) { // unit -> supernova (z-ordered), observation range, parameters
            const long long pos = pos0 + tid;
            const int si = (int)(pos / P.n_samples);
            const int ks = (int)(pos - (long long)si * P.n_samples);
            const int sn = P.perm ? __ldg(P.perm + si) : si;
            NUnit t;
            t.sn = sn;
            t.unit = sn * P.n_samples + ks;
            t.o_lo = __ldg(P.obs_offset + sn);
            t.n = __ldg(P.obs_offset + sn + 1) - t.o_lo;
            if (P.live != nullptr && __ldg(P.live + t.unit) == 0) t.n = 0; // stopped lane: nothing to evaluate
            t.z = __ldg(P.z + sn);
            t.x0 = __ldg(P.x0 + t.unit);
            t.x1 = __ldg(P.x1 + t.unit);
            t.c = __ldg(P.c + t.unit);
            t.t0 = __ldg(P.t0 + t.unit);
            units[tid] = t;
        }
        if (tid == 0) { misc[3] = 0; misc[4] = 0; }
        // ---- L2 prefetch of the next group's records (one lane per unit, last warp)
        if (warp == kWarps - 1 && group + gridDim.x < n_groups) {
            const long long q0 = unit_lo(group + gridDim.x);
            const int nn = (int)(unit_lo(group + gridDim.x + 1) - q0);
            if (lane < nn) {
                const long long pos = q0 + lane;
                const int si = (int)(pos / P.n_samples);
                const int sn = P.perm ? __ldg(P.perm + si) : si;
                const int o_lo = __ldg(P.obs_offset + sn), n = __ldg(P.obs_offset + sn + 1) - o_lo;
                const long long unit = (long long)sn * P.n_samples + (pos - (long long)si * P.n_samples);
                pf(P.z + sn); pf(P.x0 + unit); pf(P.x1 + unit); pf(P.c + unit); pf(P.t0 + unit);
                if (P.geom) { pf(P.geom + (size_t)sn * n_bands); }
                for (int o = 0; o < n + 31 && n > 0; o += 32) { // one 128-byte line of every array per step
                    const int oo = o_lo + min(o, n - 1);
                    pf(P.time + oo);
                    pf(P.band + oo);
                    if (P.zp) pf(P.zp + oo);
                    if (P.flux) { pf(P.flux + oo); pf(P.fluxerr + oo); }
                }
            }
        }
        __syncthreads();

        for (;;) {
            const int cur_u = misc[3];
            __syncthreads();
            if (cur_u >= npos) break;
            // ---- round: consecutive units whose observations fit the result array (a unit larger
            // than the array is processed alone, CAP observations at a time)
            // built by warp 0, one lane per unit: an inclusive scan of the observation counts decides how many
            // units fit; the same lanes then fill in their segment's parameters
            if (warp == 0) {
                const int u0 = misc[3], off0 = misc[4];
                __syncwarp(); // every lane has read the cursor before lane 0 advances it
                const int u = u0 + lane;
                const bool have = u < npos && lane < NSL;
                const int n = have ? units[u].n - (lane == 0 ? off0 : 0) : 0;
                int incl = n;
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) {
                    const int v = __shfl_up_sync(FULL, incl, o);
                    if (lane >= o) incl += v;
                }
                const unsigned fits = __ballot_sync(FULL, have && incl <= CAP);
                const int n_fit = fits == FULL ? 32 : __ffs(~fits) - 1; // leading run of units that fit (counts >= 0: monotone)
                const bool split = n_fit == 0;      // the first unit alone exceeds the round: CAP observations of it
                const int n_seg_w = split ? 1 : n_fit;
                const int n_ev_w = split ? CAP : __shfl_sync(FULL, incl, max(n_fit - 1, 0));
                if (lane == 0) {
                    misc[1] = n_seg_w; misc[2] = n_ev_w;
                    misc[3] = split ? u0 : u0 + n_fit;
                    misc[4] = split ? off0 + CAP : 0;
                }
                if (lane < n_seg_w) {
                    NSeg &S = segs[lane];
                    const NUnit t = units[u];
                    const int off = lane == 0 ? off0 : 0;
                    const int ks = t.unit - t.sn * P.n_samples;
                    S.n = split ? CAP : n;
                    S.e_begin = split ? 0 : incl - n;
                    S.first = off == 0;
                    S.last = split ? 0 : 1;
                    S.unit = t.unit;
                    S.sn = t.sn;
                    S.o_lo = t.o_lo + off;
                    S.out_base = (long long)t.o_lo * P.n_samples + (long long)ks * t.n + off;
                    const double cc = (double)t.c;
                    S.opz = 1.0 + (double)t.z;
                    S.inv_opz = 1.0 / S.opz;
                    S.x0 = (double)t.x0;
                    S.x1 = t.x1;
                    S.t0 = (double)t.t0;
                    S.cc = cc;
                    const double cscale = cc * 1.4426950408889634; // exponent in log2 units (ex2)
#pragma unroll
                    for (int q = 0; q < SB_MAX_CL; ++q) S.cl[q] = (float)(mp.cl[q] * cscale);
                    S.s_lo = (float)(mp.s_lo * cscale);
                    S.s_hi = (float)(mp.s_hi * cscale);
                    S.cs = (float)cscale;
                }
            }
            for (int i = tid; i < kBins; i += kThreads) hist[i] = 0;
            if (tid < kMaxBands) { win_all[tid] = 0x7fffffff; win_all[kMaxBands + tid] = -0x7fffffff; }
            for (int e = tid; e < CAP; e += kThreads) { // results of observations outside the grid stay 0
                res[e] = 0.f;
                if (GRAD) { res[CAP + e] = 0.f; res[2 * CAP + e] = 0.f; res[3 * CAP + e] = 0.f; }
            }
            __syncthreads();
            const int n_seg = misc[1], n_ev = misc[2];
            SB_CHECK(n_seg >= 1 && n_seg <= NSL && n_ev >= 0 && n_ev <= CAP);

            // ---- a1: every observation once: phase -> (rb, row weights); counting sort by (band, rb)
            float4 rec_w[KPT], rec_d[GRAD ? KPT : 1];
            int rec_key[KPT];                 // bin, or -1
            int rec_sr[KPT];                  // segment | rb << 8
            int rec_b[KPT];                   // band of the observation
            float rec_t[KPT];                 // its time
            // first pass: segment of every observation of this thread and its global loads, all in flight at once
#pragma unroll
            for (int k = 0; k < KPT; ++k) {
                const int e = tid + k * kThreads;
                rec_key[k] = -1;
                rec_sr[k] = 0;
                rec_b[k] = -1;
                rec_t[k] = 0.f;
                rec_w[k] = make_float4(0.f, 0.f, 0.f, 0.f);
                if (GRAD) rec_d[k] = make_float4(0.f, 0.f, 0.f, 0.f);
                if (e < n_ev) {
                    int lo = 0, hi = n_seg - 1; // segment of e
                    while (lo < hi) {
                        const int mid = (lo + hi + 1) >> 1;
                        if (segs[mid].e_begin <= e) lo = mid;
                        else hi = mid - 1;
                    }
                    const int o = segs[lo].o_lo + (e - segs[lo].e_begin);
                    rec_sr[k] = lo;
                    rec_b[k] = __ldg(P.band + o);
                    rec_t[k] = __ldg(P.time + o);
                }
            }
#pragma unroll
            for (int k = 0; k < KPT; ++k) {
                const int e = tid + k * kThreads;
                if (e < n_ev) {
                    const int lo = rec_sr[k];
                    const NSeg &S = segs[lo];
                    const int b = rec_b[k];
                    if ((unsigned)b < (unsigned)n_bands) {
                        int rb;
                        double wrow[4], drow[4];
                        if (obs_phase(mp, S, rec_t[k], rb, wrow, drow)) {
                            const int key = b * nq + (rb * nq) / (nP - 3);
                            SB_CHECK(rb >= 0 && rb <= nP - 4 && key >= 0 && key < kBins);
                            atomicAdd(&hist[key], 1);
                            rec_key[k] = key;
                            rec_sr[k] = lo | (rb << 8);
                            float wsl[4], wdl[4]; // register slot s holds the row congruent to s mod 4
#pragma unroll
                            for (int s = 0; s < 4; ++s) {
                                const int kk = (s - rb) & 3;
                                wsl[s] = (float)(kk == 0 ? wrow[0] : kk == 1 ? wrow[1] : kk == 2 ? wrow[2] : wrow[3]);
                                wdl[s] = (float)(kk == 0 ? drow[0] : kk == 1 ? drow[1] : kk == 2 ? drow[2] : drow[3]);
                            }
                            rec_w[k] = make_float4(wsl[0], wsl[1], wsl[2], wsl[3]);
                            if (GRAD) rec_d[k] = make_float4(wdl[0], wdl[1], wdl[2], wdl[3]);
                        }
                    }
                }
            }
            // ---- geometry of every item (band, segment) of the round: from the pack or computed here
            for (int it = tid; it < n_bands * n_seg; it += kThreads) {
                const int b = it / n_seg, sg = it - b * n_seg;
                NItem &I = items_all[it];
                if (segs[sg].n <= 0) {
                    I.n_in = 0; I.n_lo = 0; I.n_end = 0;
                } else if (P.geom) {
                    const float4 *src = reinterpret_cast<const float4 *>(P.geom + (size_t)segs[sg].sn * n_bands + b);
                    float4 *dst = reinterpret_cast<float4 *>(&I);
                    dst[0] = __ldg(src); dst[1] = __ldg(src + 1); dst[2] = __ldg(src + 2); dst[3] = __ldg(src + 3);
                } else {
                    item_geometry(mp, BV, segs[sg].opz, b, I);
                }
            }
            __syncthreads();
            // exclusive scan of the bins (all threads: kBins / kThreads bins each); start of every band's run
            {
                constexpr int PER = kBins / kThreads;
                int c[PER], s = 0;
#pragma unroll
                for (int k = 0; k < PER; ++k) { c[k] = hist[tid * PER + k]; s += c[k]; }
                int incl = s;
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) {
                    const int v = __shfl_up_sync(FULL, incl, o);
                    if (lane >= o) incl += v;
                }
                if (lane == 31) wsum[warp] = incl;
                __syncthreads();
                int run = incl - s;
                for (int w = 0; w < warp; ++w) run += wsum[w];
#pragma unroll
                for (int k = 0; k < PER; ++k) {
                    const int bin = tid * PER + k;
                    hist[bin] = run;
                    if (bin % nq == 0 && bin / nq < n_bands) bstart[bin / nq] = run;
                    run += c[k];
                }
                if (tid == kThreads - 1) bstart[n_bands] = run; // bins past n_bands * nq are empty
            }
            __syncthreads();
            const int bps = max(1, NSL / n_seg); // bands per stage
#pragma unroll
            for (int k = 0; k < KPT; ++k) { // scatter the records to their sorted positions
                if (rec_key[k] < 0) continue;
                const int e = tid + k * kThreads;
                const int sg = rec_sr[k] & 255, rb = rec_sr[k] >> 8;
                const int b = rec_key[k] / nq;
                const int slot = (b % bps) * n_seg + sg; // item slot inside the band's stage
                const int pos = atomicAdd(&hist[rec_key[k]], 1);
                SB_CHECK(pos >= 0 && pos < n_ev && n_ev <= CAP && slot >= 0 && slot < NSL && sg < n_seg && e < n_ev);
                s_ws[pos] = rec_w[k];
                if (GRAD) s_ws[CAP + pos] = rec_d[k];
                s_info[pos] = (uint32_t)slot | ((uint32_t)rb << 5) | ((uint32_t)e << 17);
            }
            // union node window of every band that has observations
            for (int it = tid; it < n_bands * n_seg; it += kThreads) {
                const int b = it / n_seg;
                NItem &I = items_all[it];
                if (bstart[b + 1] <= bstart[b]) { I.n_in = 0; I.n_lo = 0; I.n_end = 0; } // band without observations
                if (I.n_in > 0) {
                    atomicMin(&win_all[b], I.n_lo & ~3); // multiple of 4: 16-byte aligned row loads
                    atomicMax(&win_all[kMaxBands + b], I.n_end);
                }
            }
            if (tid < NSL) {
                const int bl = tid / n_seg, sg = tid - bl * n_seg;
                const float x = segs[sg].x1;
                s_x1[tid] = make_float2(x, x);
                slot_tab[tid] = bl | (sg << 8);
            }
            __syncthreads(); // sorted records, items and band windows are visible

            // ---- stages: bps bands x one 256-node window segment; phase A of stage s+1 and phase B of
            // stage s share a super-step (double-buffered node weights), one CTA barrier per stage
            const int n_bst = (n_bands + bps - 1) / bps;
            auto win_len = [&](int b) { // nodes of band b's union window (0: none)
                const int lo = win_all[b], hi = win_all[kMaxBands + b];
                return hi > lo ? hi - lo : 0;
            };
            auto n_wseg_of = [&](int st) { // window segments of band stage st (the widest band decides)
                const int b0 = st * bps, nbs = min(bps, n_bands - b0);
                int n = 0;
                for (int bl = 0; bl < nbs; ++bl) {
                    const int len = win_len(b0 + bl);
                    if (len > 0) n = max(n, (len + kSlotW - 1) / kSlotW);
                }
                return n;
            };
            // stage cursors (band stage, window segment), identical in every thread: `nxt` is the stage whose
            // node weights are built (into buffer `buf`), `cur` the one whose observations are contracted
            int st_n = 0, ws_n = 0, nws_n = 0, st_c = n_bst, ws_c = 0;
            while (st_n < n_bst && (nws_n = n_wseg_of(st_n)) == 0) ++st_n;
            int buf = 0;
            // A super-step of a warp is three tasks: its (up to) two items of phase A and its chunk of phase B.
            // Where the chunk sits among them depends on the warp: first / middle / last / middle in the four
            // warps of a scheduler, so that both kinds of work are in flight on every scheduler (the measured
            // best of four orders)
            const int wsch = (warp >> 2) & 3; // index of the warp among the warps of its scheduler
            const int bpos = wsch == 0 ? 0 : wsch == 2 ? 2 : 1;
            while (st_n < n_bst || st_c < n_bst) {
#pragma unroll 1
                for (int task = 0; task < 3; ++task) {
                    if (task != bpos) {
                        const int slice = task < bpos ? task : task - 1; // first or second item of this warp
                        // ---- phase A of stage (st_n, ws_n): node weights of its items -> buffer buf
                        if (st_n >= n_bst) continue;
                        const uint32_t at_buf = a_at + (uint32_t)(buf * BUF) * 4u;
                        const int b0 = st_n * bps, nbs = min(bps, n_bands - b0), n_items = nbs * n_seg;
                        for (int it = warp + slice * kWarps; it < n_items; it += 2 * kWarps) {
                            const int tb = slot_tab[it];
                            const int bl = tb & 255, sg = tb >> 8;
                            const int w_lo = win_all[b0 + bl], len = win_len(b0 + bl);
                            if (len <= 0) continue;
                            const int np_b = (len + 31) >> 5;
                            const int q_lo = ws_n * kPassSeg, q_hi = min(q_lo + kPassSeg, np_b);
                            if (q_lo >= q_hi) continue;
                            SB_CHECK(it < NSL && sg < n_seg && b0 + bl < n_bands && b0 * n_seg + it < n_bands * NSL);
                            phase_a_item<NCL, GRAD, NU>(mp, segs[sg], items_all[b0 * n_seg + it], w_lo, q_lo, q_hi, a_w,
                                                    at_buf + (uint32_t)(it * ATS) * 4u, lane);
                        }
                    } else {
                        // ---- phase B of stage (st_c, ws_c): its observations x buffer buf ^ 1
                        if (st_c >= n_bst) continue;
                        const uint32_t at_buf = a_at + (uint32_t)((buf ^ 1) * BUF) * 4u;
                        const int b0 = st_c * bps, nbs = min(bps, n_bands - b0);
                        for (int bl = 0; bl < nbs; ++bl) {
                            const int w_lo = win_all[b0 + bl], len = win_len(b0 + bl);
                            if (len <= 0) continue;
                            const int width = min(kSlotW, len - ws_c * kSlotW);
                            if (width <= 0) continue;
                            const int lo = bstart[b0 + bl], n = bstart[b0 + bl + 1] - lo;
                            if (n <= 0) continue;
                            const int per = (((n + kWarps - 1) / kWarps) + (GRAD ? 3 : 7)) & (GRAD ? ~3 : ~7);
                            // chunk -> warp: in stages of several bands (small batches: few observations per band)
                            // rotated from band to band, starting after the warps that carry one item more in
                            // phase A, so that every warp gets chunks; one band per stage: chunk c on warp c
                            const int rot = nbs > 1 ? (nbs * n_seg + 5 * bl) & (kWarps - 1) : 0;
                            const int i_lo = lo + ((warp - rot) & (kWarps - 1)) * per, i_hi = min(i_lo + per, lo + n);
                            if (i_lo >= i_hi) continue;
                            const int n0 = w_lo + ws_c * kSlotW;
                            SB_CHECK(n0 >= -4 && n0 + width <= mp.n_wave + 4 && i_hi <= n_ev && (n0 & 3) == 0);
                            const int nb64 = (width + 63) >> 6;
                            const bool first = ws_c == 0; // first sweep of these observations: results are stored, not added
                            // slot numbers in the records are (b % bps) * n_seg + sg = bl * n_seg + sg
                            if constexpr (GRAD) {
                                for (int h0 = 0; h0 < nb64; h0 += 2) {
                                    if (h0 + 1 < nb64)
                                        phase_b_window<1, false, true>(P, n0 + 64 * h0, at_buf + 256u * h0, SA, first && h0 == 0, i_lo, i_hi, lane);
                                    else
                                        phase_b_window<0, true, true>(P, n0 + 64 * h0, at_buf + 256u * h0, SA, first && h0 == 0, i_lo, i_hi, lane);
                                }
                            } else {
                                if (nb64 == 4) phase_b_window<2, false, false>(P, n0, at_buf, SA, first, i_lo, i_hi, lane);
                                else if (nb64 == 3) phase_b_window<1, true, false>(P, n0, at_buf, SA, first, i_lo, i_hi, lane);
                                else phase_b_window<1, false, false>(P, n0, at_buf, SA, first, i_lo, i_hi, lane);
                            }
                        }
                    }
                }
                __syncthreads();
                st_c = st_n; ws_c = ws_n; buf ^= 1;
                if (st_n < n_bst && ++ws_n >= nws_n) { // advance the build cursor
                    ws_n = 0;
                    ++st_n;
                    while (st_n < n_bst && (nws_n = n_wseg_of(st_n)) == 0) ++st_n;
                }
            }

            // ---- epilogue: one warp per segment; a6 zero point (fp64), flux [, gradient] out (coalesced),
            // a7 chi^2 [, a8 d chi^2/d theta = -2 sum (f - m)/sigma^2 dm/dtheta] in a fixed order
            float zp_last = __int_as_float(0x7fc00000); // NaN: never equal
            double zp_pow = 1.0;
            for (int sg = warp; sg < n_seg; sg += kWarps) {
                const NSeg &S = segs[sg];
                constexpr int NS = GRAD ? 5 : 1;
                double sum[NS];
#pragma unroll
                for (int k = 0; k < NS; ++k) sum[k] = 0.0;
                // four observations per lane at a time: their global loads are issued together (one latency),
                // then the arithmetic in the order of the observations (the sums keep their fixed order)
                for (int i0 = lane; i0 < S.n; i0 += 128) {
                    int b4[4];
                    float zp4[4], f4[4], e4[4];
#pragma unroll
                    for (int j = 0; j < 4; ++j) {
                        const int i = i0 + 32 * j;
                        b4[j] = -1; zp4[j] = 0.f; f4[j] = 0.f; e4[j] = 1.f;
                        if (i < S.n) {
                            const int o = S.o_lo + i;
                            b4[j] = __ldg(P.band + o);
                            if (P.zp != nullptr) zp4[j] = __ldg(P.zp + o);
                            if (want_chi) { f4[j] = __ldg(P.flux + o); e4[j] = __ldg(P.fluxerr + o); }
                        }
                    }
#pragma unroll
                    for (int j = 0; j < 4; ++j) {
                        const int i = i0 + 32 * j;
                        if (i >= S.n) break;
                        const int b = b4[j];
                        const double qnan = __longlong_as_double(0x7ff8000000000000LL);
                        double m = qnan, dm[4] = {qnan, qnan, qnan, qnan};
                        if ((unsigned)b < (unsigned)P.n_bands) {
                            double sc = 1.0;
                            if (P.zp != nullptr) { // 10^(0.4 zp): recomputed only when zp changes (usually never)
                                const float zpv = zp4[j];
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
                            const double f = (double)f4[j], e = (double)e4[j];
                            const double qv = (f - m) / e;
                            sum[0] += qv * qv;
                            if (GRAD) {
                                const double g = -2.0 * (f - m) / (e * e);
#pragma unroll
                                for (int k = 0; k < 4; ++k) sum[1 + k] += g * dm[k];
                            }
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

// ---- pack: item geometry of every (supernova, band), one thread per item -------------------------
__global__ void __launch_bounds__(256) sb_geom_kernel(SbModelParams mp, NBandsView B, const float *__restrict__ z, int n_sn,
                                                      NItem *__restrict__ geom)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= (long long)n_sn * B.n_bands) return;
    const int sn = (int)(i / B.n_bands), b = (int)(i - (long long)sn * B.n_bands);
    NItem I;
    item_geometry(mp, B, 1.0 + (double)__ldg(z + sn), b, I);
    geom[i] = I;
}

} // namespace sbn
