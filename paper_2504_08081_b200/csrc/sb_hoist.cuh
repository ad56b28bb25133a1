// sb_hoist.cuh -- the band-grouped ("hoisted") fused SALT3 band-flux kernel (sm_100a), fp32 forward.
//
// Same arithmetic per evaluation as sb_kernels.cuh, but the work
// item is one (unit, band): the observations of a unit that share a band share the rest-frame
// wavelength geometry and the colour factor (they depend on z, c and the band only -- PAPER.md:19-23,
// 38-43), so those are computed once per band sample and reused by up to kOB observations
// (G_geom = G_col = observations per (unit, band), up to 8 per pass).
//
// Mapping.  Persistent CTAs (one per SM, 16 warps) pull GROUPS of units that are neighbours in
// redshift (the z-order permutation is built by sb_zorder_kernel in the same call), and inside a group
// warps pull ITEMS (band, unit) in band-major order, so that at any time all warps of an SM read the
// same ~(71 rows x 240 columns) window of the M0/M1 table: it stays in L1 and HBM/L2 see only the
// per-observation records.  Inside an item a LANE owns one model cell per pass (29 cells per pass):
//   a2  the lane loads its node of the 4 phase rows of {M0, M1} (one coalesced LDG.64 per row of the
//       interleaved table), collapses them with the observation's phase weights (8 FFMA), gets the 3
//       neighbouring nodes by warp shuffles and converts them to the cell's cubic in tau in [0,1)
//       (Catmull-Rom = Keys a = -1/2; linear in the border cells, reading G2).  The coefficients of up
//       to 8 observations stay in REGISTERS: no row buffer, no gathers.
//   a1/a3/a4  the lane walks the 2-5 band samples that fall into its cell: tau and the reduced
//       wavelength advance by constant steps, the colour factor exp(c CL) (one ex2) times the folded
//       weight W_j (one LDS) is computed once and shared by the observations;
//   a5  per observation 3 FFMA (Horner) + 1 FFMA (accumulate); warp butterfly at the end;
//   a6/a7  epilogue per unit in fp64: zero point, flux store (coalesced), chi^2 in a fixed order.
// Requirements (checked by the host, otherwise sb_kernels.cuh runs): fp32, forward only, every band
// grid uniform, n_phase >= 4, n_wave + 48 <= LDN, n_cl <= NCL, band weights fit in shared memory.
#pragma once
#include "sb_internal.h"
#include "sb_kernels.cuh"

namespace sbh {

constexpr int kWarps = 16;
constexpr int kThreads = kWarps * 32;
constexpr int kMaxSeg = 32;  // segments (units) per round
constexpr int kOB = 8;       // observations sharing one pass
constexpr int kZBins = 512;  // redshift bins of the z-order permutation

// One segment = a contiguous run of observations of one unit (a whole unit unless it exceeds the
// round capacity); lives in shared memory for the duration of a round.
struct HSeg {
    double x0, t0, opz, inv_opz, cc;
    long long out_base;  // out_flux index of the segment's first observation
    int32_t unit;        // global unit index (supernova * n_samples + sample)
    int32_t sn;
    int32_t o_lo;        // first global observation index of the segment
    int32_t n;           // observations in the segment
    int32_t e_begin;     // first slot in the round's result array
    int32_t first, last; // first / last segment of its unit
    float x1;
    float cl[SB_MAX_CL]; // colour-law coefficients times c*log2(e)
    float s_lo, s_hi;    // continuation slopes, same scaling
    float p_lo, p_hi;    // polynomial value at the range ends, same scaling
};

struct HUnitTmp {
    int32_t unit, sn, o_lo, n;
};

struct WScratch {
    int32_t queue[64];   // observations of the item waiting for a chunk
};

struct HSmem {
    size_t w, res, segs, utmp, scr, misc, total;
    __host__ __device__ HSmem(int n_band_total, int cap)
    {
        size_t o = 0;
        w = o; o += (size_t)((n_band_total + 3) & ~3) * sizeof(float);
        res = o; o += (size_t)((cap + 3) & ~3) * sizeof(float);
        o = (o + 15) & ~(size_t)15;
        segs = o; o += (size_t)kMaxSeg * sizeof(HSeg);
        utmp = o; o += (size_t)kMaxSeg * sizeof(HUnitTmp);
        scr = o; o += (size_t)kWarps * sizeof(WScratch);
        misc = o; o += 64;
        total = o;
    }
};

// ---- z-order permutation: STABLE counting sort of the supernovae by 1/(1+z), two small kernels -----
// The supernovae are cut into kZSegs contiguous segments, one per warp (kZCtas CTAs of kZWarps warps).
// sb_zhist_kernel counts the bins of every segment (ranks inside a warp step come from
// __match_any_sync, counters are warp private) into hist[segment][bin] and adds them to tot[bin];
// sb_zscatter_kernel turns tot into bin offsets, adds the counts of the lower segments and scatters.
// The permutation is stable, hence the same on every run: the groups of the tiled kernel, and with them
// its rounding order, are reproducible.  Workspace: tot[kZBins] (zeroed by the caller), hist.
constexpr int kZWarps = 8;
constexpr int kZCtas = 32;
constexpr int kZSegs = kZWarps * kZCtas;

__device__ __forceinline__ int z_bin(const float *__restrict__ z, int i)
{
    const float key = 1.0f / (1.0f + __ldg(z + i)); // window position scales with 1/(1+z)
    int b = (int)(key * (float)kZBins);
    if (!(key > 0.0f)) b = 0;
    return min(max(b, 0), kZBins - 1);
}
__device__ __forceinline__ int z_chunk(int n_sn) { return (((n_sn + kZSegs - 1) / kZSegs) + 31) & ~31; }

__global__ void __launch_bounds__(kZWarps * 32, 1) sb_zhist_kernel(const float *__restrict__ z, int n_sn, uint32_t *hist,
                                                                   uint32_t *tot, unsigned int *counter)
{
    constexpr unsigned FULL = 0xffffffffu;
    __shared__ uint32_t cnt[kZWarps][kZBins]; // 16 KB
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (blockIdx.x == 0 && tid == 0) *counter = 0u; // group counter of the main kernel
    for (int i = tid; i < kZWarps * kZBins; i += kZWarps * 32) (&cnt[0][0])[i] = 0u;
    __syncthreads();
    const int seg = blockIdx.x * kZWarps + warp, chunk = z_chunk(n_sn);
    const int lo = min(seg * chunk, n_sn), hi = min(lo + chunk, n_sn);
    constexpr int U = 4; // steps whose loads are in flight together
    uint32_t *mine = cnt[warp];
    for (int i0 = lo; i0 < hi; i0 += 32 * U) {
        int bn[U];
#pragma unroll
        for (int u = 0; u < U; ++u) bn[u] = i0 + 32 * u + lane < hi ? z_bin(z, i0 + 32 * u + lane) : -1;
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const unsigned m = __match_any_sync(FULL, bn[u]);
            if (bn[u] >= 0 && lane == __ffs(m) - 1) mine[bn[u]] += (uint32_t)__popc(m);
            __syncwarp();
        }
    }
    __syncthreads();
    for (int i = tid; i < kZWarps * kZBins; i += kZWarps * 32) {
        const int w = i / kZBins, b = i - w * kZBins;
        const uint32_t c = cnt[w][b];
        hist[(size_t)(blockIdx.x * kZWarps + w) * kZBins + b] = c;
        if (c) atomicAdd(tot + b, c); // integer sums: order does not matter
    }
}

__global__ void __launch_bounds__(kZWarps * 32, 1) sb_zscatter_kernel(const float *__restrict__ z, int n_sn,
                                                                      const uint32_t *__restrict__ hist,
                                                                      const uint32_t *__restrict__ tot, int32_t *perm)
{
    constexpr unsigned FULL = 0xffffffffu;
    constexpr int NT = kZWarps * 32, PER = kZBins / NT; // bins per thread in the prefix steps
    __shared__ uint32_t cnt[kZWarps][kZBins];
    __shared__ uint32_t wsum[kZWarps];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    // offset of every bin: exclusive scan of tot (thread t owns bins PER t .. PER t + PER - 1)
    uint32_t bt[PER], run = 0;
#pragma unroll
    for (int k = 0; k < PER; ++k) { bt[k] = tot[tid * PER + k]; run += bt[k]; }
    uint32_t incl = run;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const uint32_t v = __shfl_up_sync(FULL, incl, o);
        if (lane >= o) incl += v;
    }
    if (lane == 31) wsum[warp] = incl;
    __syncthreads();
    uint32_t base = incl - run;
    for (int w = 0; w < warp; ++w) base += wsum[w];
    // plus the counts of all lower segments, then of the lower warps of this CTA
    const int seg0 = blockIdx.x * kZWarps;
#pragma unroll
    for (int k = 0; k < PER; ++k) {
        const int b = tid * PER + k;
        uint32_t a = base;
        for (int sgm = 0; sgm < seg0; ++sgm) a += hist[(size_t)sgm * kZBins + b];
        for (int w = 0; w < kZWarps; ++w) {
            cnt[w][b] = a;
            a += hist[(size_t)(seg0 + w) * kZBins + b];
        }
        base += bt[k];
    }
    __syncthreads();
    const int seg = seg0 + warp, chunk = z_chunk(n_sn);
    const int lo = min(seg * chunk, n_sn), hi = min(lo + chunk, n_sn);
    constexpr int U = 4;
    uint32_t *mine = cnt[warp];
    for (int i0 = lo; i0 < hi; i0 += 32 * U) {
        int bn[U];
#pragma unroll
        for (int u = 0; u < U; ++u) bn[u] = i0 + 32 * u + lane < hi ? z_bin(z, i0 + 32 * u + lane) : -1;
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const unsigned m = __match_any_sync(FULL, bn[u]);
            const uint32_t at = bn[u] >= 0 ? mine[bn[u]] : 0u;
            __syncwarp();
            if (bn[u] >= 0 && lane == __ffs(m) - 1) mine[bn[u]] = at + (uint32_t)__popc(m);
            __syncwarp();
            if (bn[u] >= 0) perm[at + (uint32_t)__popc(m & ((1u << lane) - 1u))] = i0 + 32 * u + lane;
        }
    }
}

// Small batches (n_sn <= kZSmall): the same stable sort in ONE CTA of 16 warps (no workspace, no memset,
// one launch instead of two): warp w owns a contiguous range and a private counter row.
constexpr int kZSmall = 8192;
__global__ void __launch_bounds__(512, 1) sb_zorder_small_kernel(const float *__restrict__ z, int n_sn, int32_t *perm,
                                                                 unsigned int *counter)
{
    constexpr unsigned FULL = 0xffffffffu;
    constexpr int NWZ = 16;
    __shared__ uint32_t cnt[NWZ][kZBins]; // 32 KB
    __shared__ uint32_t wsum[NWZ];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid == 0) *counter = 0u;
    for (int i = tid; i < NWZ * kZBins; i += NWZ * 32) (&cnt[0][0])[i] = 0u;
    __syncthreads();
    const int chunk = (((n_sn + NWZ - 1) / NWZ) + 31) & ~31;
    const int lo = min(warp * chunk, n_sn), hi = min(lo + chunk, n_sn);
    uint32_t *mine = cnt[warp];
    for (int i0 = lo; i0 < hi; i0 += 32) {
        const int bn = i0 + lane < hi ? z_bin(z, i0 + lane) : -1;
        const unsigned m = __match_any_sync(FULL, bn);
        if (bn >= 0 && lane == __ffs(m) - 1) mine[bn] += (uint32_t)__popc(m);
        __syncwarp();
    }
    __syncthreads();
    { // bin t: exclusive prefix over the warps, then over the bins (NWZ * 32 == kZBins threads)
        const int t = tid;
        uint32_t s = 0;
#pragma unroll
        for (int w = 0; w < NWZ; ++w) {
            const uint32_t c = cnt[w][t];
            cnt[w][t] = s;
            s += c;
        }
        uint32_t incl = s;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t v = __shfl_up_sync(FULL, incl, o);
            if (lane >= o) incl += v;
        }
        if (lane == 31) wsum[warp] = incl;
        __syncthreads();
        uint32_t base = incl - s;
        for (int w = 0; w < warp; ++w) base += wsum[w];
#pragma unroll
        for (int w = 0; w < NWZ; ++w) cnt[w][t] += base;
    }
    __syncthreads();
    for (int i0 = lo; i0 < hi; i0 += 32) {
        const int bn = i0 + lane < hi ? z_bin(z, i0 + lane) : -1;
        const unsigned m = __match_any_sync(FULL, bn);
        const uint32_t at = bn >= 0 ? mine[bn] : 0u;
        __syncwarp();
        if (bn >= 0 && lane == __ffs(m) - 1) mine[bn] = at + (uint32_t)__popc(m);
        __syncwarp();
        if (bn >= 0) perm[at + (uint32_t)__popc(m & ((1u << lane) - 1u))] = i0 + lane;
    }
}
static_assert(kZBins == 512, "sb_zorder_small_kernel: one thread per bin");

// ---- colour law of one item: exponent argument (log2 units) as a function of the reduced wavelength
template <int NCL> struct HColour {
    float a[NCL];
    float r_lo, r_hi, s_lo, s_hi;
    float lin_a, lin_b; // CM_LINEAR: arg = lin_a + lin_b * r
    template <int CM> __device__ __forceinline__ float arg(float r) const
    {
        if constexpr (CM == sb::CM_LINEAR) {
            return __fmaf_rn(r, lin_b, lin_a);
        } else if constexpr (CM == sb::CM_INSIDE) {
            float p = a[NCL - 1];
#pragma unroll
            for (int q = NCL - 2; q >= 0; --q) p = __fmaf_rn(p, r, a[q]);
            return p;
        } else {
            const float rc = fminf(fmaxf(r, r_lo), r_hi);
            const float d = r - rc;
            const float slope = d > 0.0f ? s_hi : s_lo;
            float p = a[NCL - 1];
#pragma unroll
            for (int q = NCL - 2; q >= 0; --q) p = __fmaf_rn(p, rc, a[q]);
            return __fmaf_rn(slope, d, p);
        }
    }
    // the same for two wavelengths at once, as packed FP32 pairs (one issue slot per pair of FMAs)
    template <int CM> __device__ __forceinline__ float2 arg2(float2 r) const
    {
        if constexpr (CM == sb::CM_LINEAR) {
            return __ffma2_rn(r, make_float2(lin_b, lin_b), make_float2(lin_a, lin_a));
        } else if constexpr (CM == sb::CM_INSIDE) {
            float2 p = make_float2(a[NCL - 1], a[NCL - 1]);
#pragma unroll
            for (int q = NCL - 2; q >= 0; --q) p = __ffma2_rn(p, r, make_float2(a[q], a[q]));
            return p;
        } else {
            const float2 rc = make_float2(fminf(fmaxf(r.x, r_lo), r_hi), fminf(fmaxf(r.y, r_lo), r_hi));
            const float2 d = make_float2(r.x - rc.x, r.y - rc.y);
            const float2 slope = make_float2(d.x > 0.0f ? s_hi : s_lo, d.y > 0.0f ? s_hi : s_lo);
            float2 p = make_float2(a[NCL - 1], a[NCL - 1]);
#pragma unroll
            for (int q = NCL - 2; q >= 0; --q) p = __ffma2_rn(p, rc, make_float2(a[q], a[q]));
            return __ffma2_rn(slope, d, p);
        }
    }
};

// Geometry of one item (unit, band): warp-uniform values.
struct HGeo {
    int32_t n_in;     // in-range band samples
    int32_t ncell;    // model cells spanned
    int32_t g_first;  // first cell
    int32_t wbase;    // index of the first in-range sample in the staged weight table
    int32_t cmode;
    float c0;         // u of the first in-range sample minus g_first
    float ha_hi, ha_lo, inv_ha; // cells per band sample (split in two floats), its inverse
    float hal, r_first;         // reduced-wavelength step per sample, value at the first sample
};

// Sum NV values per lane across the warp so that lane L ends with the total of value (L >> SH),
// SH = 5 - log2(NV): log2(NV) halving steps (each lane keeps the half selected by one lane bit and
// sends the other half to its partner), then plain butterflies over the remaining lane bits.
template <int NV> __device__ __forceinline__ float warp_reduce_transpose(float (&v)[NV], int lane)
{
    constexpr unsigned FULL = 0xffffffffu;
    static_assert(NV == 4 || NV == 8 || NV == 16 || NV == 32, "NV must be a power of two in [4, 32]");
    int mask = 16;
#pragma unroll
    for (int n = NV; n > 1; n >>= 1) {
        const bool hi = (lane & mask) != 0;
#pragma unroll
        for (int i = 0; i < n / 2; ++i) {
            const float keep = hi ? v[i + n / 2] : v[i];
            const float send = hi ? v[i] : v[i + n / 2];
            v[i] = keep + __shfl_xor_sync(FULL, send, mask);
        }
        mask >>= 1;
    }
    float r = v[0];
#pragma unroll
    for (int m = 16 / NV; m > 0; m >>= 1) r += __shfl_xor_sync(FULL, r, m);
    return r;
}

// One chunk: up to NOB (a power of two) observations of the item integrated together; n valid.
//
// The band integral of observation o is  sum_j ew_j sum_m w_m(tau_j) R_o[i_j + m]  (R_o = the
// phase-collapsed row, w_m = Keys weights, ew_j = colour factor x folded band weight).  Exchanging the
// sums (an exact re-association) gives  sum_l At[l] R_o[l]  with the NODE WEIGHTS
// At[l] = sum_j ew_j w_{l - i_j}(tau_j), which do not depend on the observation: they are built once
// per chunk from the per-cell moments sum ew tau^p, and every observation then costs 8 FFMA per model
// node (4 phase rows x {M0, M1}) with the phase weights applied after the warp reduction.
template <int NOB, int NCL, int LDN>
__device__ __forceinline__ void run_chunk(int n, const SbHParams &P, const HSeg &S, const HGeo &G,
                                          const HColour<NCL> &col, WScratch &W, const float *__restrict__ s_w,
                                          float *__restrict__ res, int lane)
{
    constexpr unsigned FULL = 0xffffffffu;
    constexpr int ROWB = LDN * (int)sizeof(float2); // bytes per phase row (compile time: immediate offsets)
    constexpr int NV = 4 * NOB;                     // accumulators per lane: D[o][k], k = phase row
    constexpr int SH = NV == 32 ? 0 : NV == 16 ? 1 : NV == 8 ? 2 : 3; // lane -> value index shift
    const SbModelParams &mp = P.mp;
    const int nW = mp.n_wave, nP = mp.n_phase;

    // ---- a1/a2 per observation: lane (o, k) = ((lane >> SH) >> 2, (lane >> SH) & 3) holds the weight
    // of phase row rb + k of observation o; everything scalar per observation is fp64
    const int my_o = (lane >> SH) >> 2, my_k = (lane >> SH) & 3;
    float my_w = 0.f;
    int my_rowoff = 0, my_slot = -1;
    if (my_o < n) {
        const int oi = W.queue[my_o];
        const int o = S.o_lo + oi;
        const double p = ((double)__ldg(P.time + o) - S.t0) * S.inv_opz;
        const double up = (p - mp.p0) / mp.dp;
        int kp = 0;
        double wv[4] = {0.0, 0.0, 0.0, 0.0}, wd[4];
        if ((up >= 0.0) && (up <= (double)(nP - 1))) { // outside the phase grid: zero flux (G3)
            kp = min((int)floor(up), nP - 2);
            sb::phase_weights(up - (double)kp, (kp == 0) || (kp == nP - 2), 1.0, wv, wd);
        }
        const int rb = min(max(kp - 1, 0), nP - 4); // rows rb..rb+3 are loaded
        const int src = my_k - ((kp - 1) - rb);     // row rb + k carries Keys weight index src
        double w = 0.0;
        if (src == 0) w = wv[0];
        if (src == 1) w = wv[1];
        if (src == 2) w = wv[2];
        if (src == 3) w = wv[3];
        my_w = (float)w;
        my_rowoff = rb * ROWB;
        my_slot = S.e_begin + oi;
    }
    int rowoff[NOB];
#pragma unroll
    for (int o = 0; o < NOB; ++o) rowoff[o] = __shfl_sync(FULL, my_rowoff, (o * 4) << SH);
    float D[NV];
#pragma unroll
    for (int i = 0; i < NV; ++i) D[i] = 0.f;

    // pass q: lane l <-> NODE column nbcol + 32 q + l of the table (a 256-byte aligned window: every
    // LDG.64 of the warp touches exactly two 128-byte lines) and <-> CELL (node + 1).  Node n takes
    // w_{-1} of cell n+1 (this lane), w_0 of cell n (lane - 1), w_1 of cell n-1 (lane - 2) and w_2 of
    // cell n-2 (lane - 3); lanes 0..2 take them from the previous pass (carried in registers).
    const int col_first = G.g_first - 1 + SBH_PAD_L;          // column of the first node needed
    const int nbcol = col_first & ~15;
    const int n_pass = (G.g_first + G.ncell + 1 + SBH_PAD_L - nbcol) / 32 + 1; // last node: g_last + 2
    const char *colp = reinterpret_cast<const char *>(P.m01) + (ptrdiff_t)(nbcol + lane) * (ptrdiff_t)sizeof(float2);
    const float c0 = G.c0, inv_ha = G.inv_ha, ha_hi = G.ha_hi, ha_lo = G.ha_lo, hal = G.hal, r_first = G.r_first;
    const int n_in = G.n_in, ncell = G.ncell;
    const float x1 = S.x1;
    auto jstart = [&](int x) { // first band sample (relative to the first in-range one) of cell x
        int j = (int)ceilf(((float)x - c0) * inv_ha);
        j = min(max(j, 0), n_in);
        if (x <= 0) j = 0;
        if (x >= ncell) j = n_in;
        return j;
    };
    constexpr int NA = NOB > 4 ? NOB / 2 : NOB; // observations whose loads are issued before the sample loop
    float pa0 = 0.f, pa1 = 0.f, pa2 = 0.f;      // w_0, w_1, w_2 of the previous pass's cells
    int gq = nbcol - SBH_PAD_L + 1 + lane - G.g_first; // this lane's cell relative to g_first

    for (int q = 0; q < n_pass; ++q) {
        // ---- a2 loads, first batch: this lane's node of the 4 phase rows ({M0, M1} pairs)
        float2 rawa[NA][4];
#pragma unroll
        for (int o = 0; o < NA; ++o) {
            const char *p = colp + rowoff[o];
#pragma unroll
            for (int k = 0; k < 4; ++k) rawa[o][k] = __ldg(reinterpret_cast<const float2 *>(p + k * ROWB));
        }

        // ---- a1: the band samples of this lane's cell
        const int js = jstart(gq), je = jstart(gq + 1);
        const int cnt = je - js;
        const float jsf = (float)js;
        float tau = __fmaf_rn(jsf, ha_lo, __fmaf_rn(jsf, ha_hi, -(float)gq)) + c0; // u_js - cell
        float r = __fmaf_rn(jsf, hal, r_first);
        const float *wp = s_w + (G.wbase + js);
        const int km = __reduce_max_sync(FULL, cnt);

        // ---- a3/a4: moments of the cell: S_p = sum_k ew_k tau_k^p
        float s0 = 0.f, s1 = 0.f, s2 = 0.f, s3 = 0.f;
        auto samples = [&](auto cm_tag) {
            constexpr int CM = decltype(cm_tag)::value;
            for (int k = 0; k < km; ++k) {
                float w = 0.f;
                if (k < cnt) w = wp[k];
                const float ew = sb::exp_scaled(col.template arg<CM>(r)) * w;
                const float t2 = tau * tau;
                s0 += ew;
                s1 = __fmaf_rn(ew, tau, s1);
                s2 = __fmaf_rn(ew, t2, s2);
                s3 = __fmaf_rn(ew, t2 * tau, s3);
                tau += ha_hi;
                r += hal;
            }
        };
        if (G.cmode == sb::CM_INSIDE) samples(std::integral_constant<int, sb::CM_INSIDE>{});
        else if (G.cmode == sb::CM_LINEAR) samples(std::integral_constant<int, sb::CM_LINEAR>{});
        else samples(std::integral_constant<int, sb::CM_GENERIC>{});

        // ---- moments -> weights on the cell's four nodes (Keys a = -1/2; linear in border cells, G2)
        const int g = G.g_first + gq;
        float am = 0.5f * (__fmaf_rn(2.0f, s2, -s3) - s1);
        float a0 = __fmaf_rn(1.5f, s3, __fmaf_rn(-2.5f, s2, s0));
        float a1 = 0.5f * (__fmaf_rn(4.0f, s2, s1) - 3.0f * s3);
        float a2 = 0.5f * (s3 - s2);
        if (g <= 0 || g >= nW - 2) {
            am = 0.f;
            a0 = s0 - s1;
            a1 = s1;
            a2 = 0.f;
        }
        // node weight of this lane's node
        auto from_left = [&](float cur, float prev, int d) {
            const float a = __shfl_up_sync(FULL, cur, d);
            const float b = __shfl_sync(FULL, prev, (lane - d) & 31);
            return lane >= d ? a : b;
        };
        const float at = am + from_left(a0, pa0, 1) + from_left(a1, pa1, 2) + from_left(a2, pa2, 3);
        pa0 = a0;
        pa1 = a1;
        pa2 = a2;
        const float at1 = at * x1;

        // ---- a2/a5: D[o][k] += At * (M0 + x1 M1)[rb_o + k][node]
        if constexpr (NOB > NA) {
            float2 rawb[NOB - NA][4];
#pragma unroll
            for (int o = NA; o < NOB; ++o) {
                const char *p = colp + rowoff[o];
#pragma unroll
                for (int k = 0; k < 4; ++k) rawb[o - NA][k] = __ldg(reinterpret_cast<const float2 *>(p + k * ROWB));
            }
#pragma unroll
            for (int o = 0; o < NA; ++o) {
#pragma unroll
                for (int k = 0; k < 4; ++k) D[o * 4 + k] = __fmaf_rn(at, rawa[o][k].x, __fmaf_rn(at1, rawa[o][k].y, D[o * 4 + k]));
            }
#pragma unroll
            for (int o = NA; o < NOB; ++o) {
#pragma unroll
                for (int k = 0; k < 4; ++k)
                    D[o * 4 + k] = __fmaf_rn(at, rawb[o - NA][k].x, __fmaf_rn(at1, rawb[o - NA][k].y, D[o * 4 + k]));
            }
        } else {
#pragma unroll
            for (int o = 0; o < NA; ++o) {
#pragma unroll
                for (int k = 0; k < 4; ++k) D[o * 4 + k] = __fmaf_rn(at, rawa[o][k].x, __fmaf_rn(at1, rawa[o][k].y, D[o * 4 + k]));
            }
        }
        colp += 32 * sizeof(float2);
        gq += 32;
    }
    // ---- a5: warp reduction (lane (o, k) ends with D[o][k]), phase weights, sum over the 4 rows
    float v = warp_reduce_transpose<NV>(D, lane) * my_w;
    v += __shfl_xor_sync(FULL, v, 1 << SH);
    v += __shfl_xor_sync(FULL, v, 2 << SH);
    if (my_slot >= 0 && my_k == 0 && (lane & ((1 << SH) - 1)) == 0) res[my_slot] = v;
    __syncwarp();
}

template <int NCL, int LDN>
__device__ __forceinline__ void run_chunk_n(int n, const SbHParams &P, const HSeg &S, const HGeo &G,
                                            const HColour<NCL> &col, WScratch &W, const float *s_w, float *res, int lane)
{
    if (n > 4) run_chunk<8, NCL, LDN>(n, P, S, G, col, W, s_w, res, lane);
    else if (n > 2) run_chunk<4, NCL, LDN>(n, P, S, G, col, W, s_w, res, lane);
    else if (n > 1) run_chunk<2, NCL, LDN>(n, P, S, G, col, W, s_w, res, lane);
    else run_chunk<1, NCL, LDN>(n, P, S, G, col, W, s_w, res, lane);
}

// One item: the observations of segment S in band b.
template <int NCL, int LDN>
__device__ __forceinline__ void run_item(const SbHParams &P, const HSeg &S, int b, WScratch &W, const float *s_w,
                                         float *res, int lane)
{
    constexpr unsigned FULL = 0xffffffffu;
    const SbModelParams &mp = P.mp;
    const int nW = mp.n_wave;
    // ---- geometry of (z, band): in-range samples decided in fp64 (G9), window of model cells
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

    HGeo G;
    const double a_d = inv_opz / mp.dl;                        // cells per observer-frame Angstrom
    const double ub = (lam_first * inv_opz - mp.l0) / mp.dl;   // u of dlam = 0
    const double ha = h * a_d;                                 // cells per band sample
    const double u_lo = (double)j_lo * ha + ub;
    const double u_hi = (double)(j_hi - 1) * ha + ub;
    const int g_first = min(max((int)floor(u_lo), 0), nW - 2);
    const int g_last = min(max((int)floor(u_hi), 0), nW - 2);
    G.n_in = j_hi - j_lo;
    G.g_first = g_first;
    G.ncell = g_last - g_first + 1;
    G.wbase = boff + j_lo;
    G.c0 = (float)(u_lo - (double)g_first);
    G.ha_hi = (float)ha;
    G.ha_lo = (float)(ha - (double)G.ha_hi);
    G.inv_ha = (float)(1.0 / ha);
    const double al_d = inv_opz * mp.cl_inv_span;
    const double be_d = (lam_first * inv_opz - mp.cl_b) * mp.cl_inv_span;
    const double hal = h * al_d;
    const double r_a = (double)j_lo * hal + be_d, r_b = (double)(j_hi - 1) * hal + be_d;
    G.hal = (float)hal;
    G.r_first = (float)r_a;
    // ---- a3: colour-law mode of the item (reduced wavelength is monotone in j)
    HColour<NCL> col;
#pragma unroll
    for (int q = 0; q < NCL; ++q) col.a[q] = S.cl[q];
    col.r_lo = (float)mp.r_lo;
    col.r_hi = (float)mp.r_hi;
    col.s_lo = S.s_lo;
    col.s_hi = S.s_hi;
    col.lin_a = 0.f;
    col.lin_b = 0.f;
    {
        const double r_min = fmin(r_a, r_b), r_max = fmax(r_a, r_b);
        const double margin = 1e-4;
        int cmode = sb::CM_GENERIC;
        if (r_min >= mp.r_lo + margin && r_max <= mp.r_hi - margin) {
            cmode = sb::CM_INSIDE;
        } else if (r_min >= mp.r_hi + margin) { // arg = p_hi + s_hi (r - r_hi)
            cmode = sb::CM_LINEAR;
            col.lin_b = S.s_hi;
            col.lin_a = (float)((double)S.p_hi - (double)S.s_hi * mp.r_hi);
        } else if (r_max <= mp.r_lo - margin) {
            cmode = sb::CM_LINEAR;
            col.lin_b = S.s_lo;
            col.lin_a = (float)((double)S.p_lo - (double)S.s_lo * mp.r_lo);
        }
        G.cmode = cmode;
    }

    // ---- the observations of this band, in order, in chunks of kOB
    int qn = 0;
    for (int base = 0; base < S.n; base += 32) {
        const int oi = base + lane;
        bool match = false;
        if (oi < S.n) match = __ldg(P.band + S.o_lo + oi) == b;
        const unsigned m = __ballot_sync(FULL, match);
        if (match) W.queue[qn + __popc(m & ((1u << lane) - 1u))] = oi;
        qn += __popc(m);
        __syncwarp();
        while (qn >= kOB) {
            run_chunk<kOB, NCL, LDN>(kOB, P, S, G, col, W, s_w, res, lane);
            const int rest = qn - kOB; // <= 31
            int v = 0;
            if (lane < rest) v = W.queue[kOB + lane];
            __syncwarp();
            if (lane < rest) W.queue[lane] = v;
            __syncwarp();
            qn = rest;
        }
    }
    if (qn > 0) run_chunk_n<NCL, LDN>(qn, P, S, G, col, W, s_w, res, lane);
}

// ---- the kernel ---------------------------------------------------------------------------------
template <int NCL, int LDN>
__global__ void __launch_bounds__(kThreads, 1) sb_hoist_kernel(const __grid_constant__ SbHParams P)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const SbModelParams &mp = P.mp;
    const HSmem L(P.n_band_total, P.cap);
    float *s_w = reinterpret_cast<float *>(smem_raw + L.w);
    float *res = reinterpret_cast<float *>(smem_raw + L.res);
    HSeg *segs = reinterpret_cast<HSeg *>(smem_raw + L.segs);
    HUnitTmp *utmp = reinterpret_cast<HUnitTmp *>(smem_raw + L.utmp);
    WScratch *scr = reinterpret_cast<WScratch *>(smem_raw + L.scr);
    int *misc = reinterpret_cast<int *>(smem_raw + L.misc);       // [0] group, [1] n_seg, [2] n_ev, [3] next unit, [4] next offset, [5] item counter
    double *carry = reinterpret_cast<double *>(smem_raw + L.misc + 32); // chi^2 of a unit split over rounds

    for (int i = tid; i < P.n_band_total; i += kThreads) s_w[i] = __ldg(P.band_w + i);
    const long long n_units = (long long)P.n_sn * P.n_samples;
    const int G = P.group_units, CAP = P.cap;
    const long long n_groups = (n_units + G - 1) / G;
    const bool want_chi = P.out_chi2 != nullptr;

    for (;;) {
        __syncthreads();
        if (tid == 0) misc[0] = (int)atomicAdd(P.counter, 1u);
        __syncthreads();
        const long long group = (long long)(unsigned)misc[0];
        if (group >= n_groups) break;
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
                while (u < npos && n_seg < kMaxSeg) {
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
                misc[1] = n_seg; misc[2] = n_ev; misc[3] = u; misc[4] = off; misc[5] = 0;
            }
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
            for (int e = tid; e < n_ev; e += kThreads) res[e] = 0.f;
            __syncthreads();

            // ---- main: warps pull items (band-major: all warps work on the same band window)
            const int n_items = P.n_bands * n_seg;
            for (;;) {
                int it = 0;
                if (lane == 0) it = atomicAdd(&misc[5], 1);
                it = __shfl_sync(0xffffffffu, it, 0);
                if (it >= n_items) break;
                const int b = it / n_seg, sg = it - b * n_seg;
                if (segs[sg].n > 0) run_item<NCL, LDN>(P, segs[sg], b, scr[warp], s_w, res, lane);
            }
            __syncthreads();

            // ---- epilogue: one warp per segment; a6 zero point (fp64), flux out (coalesced), a7 chi^2
            for (int sg = warp; sg < n_seg; sg += kWarps) {
                const HSeg &S = segs[sg];
                double sum = 0.0;
                for (int i = lane; i < S.n; i += 32) {
                    const int o = S.o_lo + i;
                    const int b = __ldg(P.band + o);
                    double m;
                    if ((unsigned)b >= (unsigned)P.n_bands) {
                        m = __longlong_as_double(0x7ff8000000000000LL);
                    } else {
                        double sc = 1.0;
                        if (P.zp != nullptr) sc = exp10(0.4 * (double)__ldg(P.zp + o)) * __ldg(P.band_zpab_inv + b);
                        m = sc * S.x0 * (double)res[S.e_begin + i];
                    }
                    if (P.out_flux) P.out_flux[S.out_base + i] = (float)m;
                    if (want_chi) {
                        const double f = (double)__ldg(P.flux + o), e = (double)__ldg(P.fluxerr + o);
                        const double qv = (f - m) / e;
                        sum += qv * qv;
                    }
                }
                if (want_chi) {
                    sum = sb::warp_sum(sum);
                    if (lane == 0) {
                        const double total = (S.first ? 0.0 : *carry) + sum;
                        if (S.last) P.out_chi2[S.unit] = (float)total;
                        else *carry = total;
                    }
                }
            }
            __syncthreads();
        }
    }
}

} // namespace sbh
