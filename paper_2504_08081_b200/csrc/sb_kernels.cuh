// sb_kernels.cuh -- the fused SALT3 band-flux kernel (sm_100a).
//
// Persistent CTAs; a CTA takes groups of G consecutive units (unit = supernova s x parameter
// sample k) and works through the group's evaluations (one per observation of each unit) in chunks
// of at most CAP:
//   prologue  one THREAD per evaluation: everything that is scalar per evaluation (fp64): phase,
//             phase weights, in-range band samples, cell window, zero point -> a record in smem.
//   main      one WARP per evaluation (dynamic, smem counter); lanes stride the band's samples.
//   epilogue  one thread per evaluation: coalesced result stores, chi^2 terms; then one warp per
//             unit reduces them in a fixed order (deterministic).
// Steps (citations in include/saltband.h):
//   a1  p = (t - t0)/(1+z) per evaluation; per sample the fractional cell coordinate relative to
//       the evaluation's first cell as ONE FFMA  t_j = dlam_j * a + b  (dlam_j = lam_j - lam_first
//       is exact in fp32).
//   a2  bicubic interpolation, separable: the <= 4 phase rows of M0 and M1 are collapsed once per
//       evaluation into a 1-D row R[l] = sum_k wp_k (M0 + x1 M1)[kp+k][l] (float4 loads: 4 nodes
//       per lane, 120 cells per warp pass, 3 shuffles for the halo); each cell of that row is
//       converted to the cubic's coefficients about the cell centre (an exact re-association of
//       the Keys a=-1/2 / Catmull-Rom weights; linear in border cells) and stored as one float4
//       per cell in this warp's shared-memory row buffer (XOR-swizzled: conflict-free stores).
//       A sample is then 1 LDS.128 + 3 FFMA.
//   a3  colour law: degree-(NCL-1) Horner in the reduced wavelength, linear continuation by
//       clamping, one ex2 per sample (coefficients pre-scaled by c*log2(e) in fp32 forward mode).
//   a4/a5  folded weight W_j = w_j T_j lam_j/(hc) (trapezoid weight folded at load), interleaved
//       with dlam_j (one LDS.64), FFMA accumulate per lane, warp-shuffle butterfly.
//   a6  zero point S = 10^(0.4 zp)/ZPAB_b in fp64 per evaluation (prologue).
//   a7  chi^2 per unit in fp64, fixed summation order.
//   a8  analytic gradient: three coefficient sets (value row, M1-only row, d/dphase row) and four
//       accumulators give d m/d(x0, x1, c, t0).
#pragma once
#include <type_traits>

#include "sb_internal.h"

namespace sb {

constexpr int kWarpSize = 32;
constexpr int kCellsPerPass = 120; // lanes 1..30 produce 4 cells each; lanes 0 and 31 carry the halo
constexpr int kMaxGroup = 16;      // units per CTA group

template <typename T> struct Vec4;
template <> struct Vec4<float> { using type = float4; };
template <> struct Vec4<double> { using type = double4; };
template <typename T> struct Vec2;
template <> struct Vec2<float> { using type = float2; };
template <> struct Vec2<double> { using type = double2; };

template <typename T> __device__ __forceinline__ typename Vec4<T>::type make_v4(T a, T b, T c, T d);
template <> __device__ __forceinline__ float4 make_v4<float>(float a, float b, float c, float d) { return make_float4(a, b, c, d); }
template <> __device__ __forceinline__ double4 make_v4<double>(double a, double b, double c, double d) { return make_double4(a, b, c, d); }

__device__ __forceinline__ float4 ldg_v4(const float *p) { return __ldg(reinterpret_cast<const float4 *>(p)); }
__device__ __forceinline__ double4 ldg_v4(const double *p)
{
    const double2 a = __ldg(reinterpret_cast<const double2 *>(p));
    const double2 b = __ldg(reinterpret_cast<const double2 *>(p) + 1);
    return make_double4(a.x, a.y, b.x, b.y);
}

__device__ __forceinline__ float fma_t(float a, float b, float c) { return __fmaf_rn(a, b, c); }
__device__ __forceinline__ double fma_t(double a, double b, double c) { return fma(a, b, c); }

// exp of a pre-scaled argument: fp32 takes log2-units (ex2.approx), fp64 natural units.
__device__ __forceinline__ float exp_scaled(float x)
{
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ double exp_scaled(double x) { return exp(x); }
template <typename T> __device__ __forceinline__ double exp_arg_scale();
template <> __device__ __forceinline__ double exp_arg_scale<float>() { return 1.4426950408889634; }
template <> __device__ __forceinline__ double exp_arg_scale<double>() { return 1.0; }

template <typename T> __device__ __forceinline__ T warp_sum(T v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// Number of j in [0, n) with f(j) < thr (or <= thr) for a non-decreasing f; one thread.
template <typename F>
__device__ __forceinline__ int count_less(int n, double thr, F f, bool or_equal)
{
    int lo = 0, hi = n;
    while (lo < hi) {
        const int mid = (lo + hi) >> 1;
        const double v = f(mid);
        const bool less = or_equal ? (v <= thr) : (v < thr);
        if (less) lo = mid + 1; else hi = mid;
    }
    return lo;
}

// Same count, warp-cooperative 32-ary search (used only when a band needs several tiles).
template <typename F, typename T>
__device__ __forceinline__ int warp_count_less(int n, T thr, int lane, F f)
{
    int lo = 0, len = n;
    while (len > 0) {
        int step = (len + kWarpSize - 1) / kWarpSize;
        int j = lo + lane * step; // probe the first element of each of 32 sub-ranges
        bool less = false;
        if (j < lo + len) less = f(j) < thr;
        unsigned m = __ballot_sync(0xffffffffu, less);
        int cnt = __popc(m); // probes 0..cnt-1 are "less": the boundary is inside sub-range cnt-1
        if (cnt == 0) return lo;
        int new_lo = lo + (cnt - 1) * step + 1; // element at the probe itself is "less"
        int new_len = min(step - 1, lo + len - new_lo);
        lo = new_lo;
        len = new_len;
    }
    return lo;
}

// Interior cell: Catmull-Rom cubic through (rm, r0, r1, r2) about the cell centre, s in [-1/2, 1/2].
template <typename T>
__device__ __forceinline__ typename Vec4<T>::type cell_coef_interior(T rm, T r0, T r1, T r2)
{
    const T s1 = r0 + r1, s2 = rm + r2, d1 = r1 - r0, d2 = r2 - rm;
    return make_v4<T>(fma_t(s1, (T)0.5625, s2 * (T)-0.0625), fma_t(d1, (T)1.375, d2 * (T)-0.125),
                      (s2 - s1) * (T)0.25, fma_t(d1, (T)-1.5, d2 * (T)0.5));
}

// General cell g of an n-node row (nodes outside the row are zero padding and never used):
//   1 <= g <= n-3 Catmull-Rom; g = 0 or n-2 linear (G2); g = -1 and g = n-1 continue the
//   adjacent border line (reached only within rounding of the grid edge); anything else is zero.
template <typename T>
__device__ __forceinline__ typename Vec4<T>::type cell_coef(int g, int n, T rm, T r0, T r1, T r2)
{
    const T h = (T)0.5;
    if (g < -1 || g > n - 1) return make_v4<T>(0, 0, 0, 0);
    if (g == -1) { T d = r2 - r1; return make_v4<T>(r1 - h * d, d, 0, 0); }
    if (g == n - 1) { T d = r0 - rm; return make_v4<T>(r0 + h * d, d, 0, 0); }
    if (g == 0 || g == n - 2) return make_v4<T>(h * (r0 + r1), r1 - r0, 0, 0);
    return cell_coef_interior<T>(rm, r0, r1, r2);
}

template <typename T>
__device__ __forceinline__ T poly3(const typename Vec4<T>::type &a, T s)
{
    return fma_t(fma_t(fma_t(a.w, s, a.z), s, a.y), s, a.x);
}

// Row-buffer slot of entry q: q ^ ((q >> 3) & 3) -- an XOR swizzle inside groups of 8 slots so that the
// four 128-bit stores of a collapse pass (lane l writes entries 4l..4l+3) are bank-conflict free.
// Cubic-convolution weights (Keys a = -1/2) and their derivatives, or the linear border pair.
__device__ __forceinline__ void phase_weights(double tau, bool border, double inv_dp, double w[4], double d[4])
{
    if (border) {
        w[0] = 0.0; w[1] = 1.0 - tau; w[2] = tau; w[3] = 0.0;
        d[0] = 0.0; d[1] = -inv_dp; d[2] = inv_dp; d[3] = 0.0;
        return;
    }
    double t2 = tau * tau, t3 = t2 * tau;
    w[0] = 0.5 * (-t3 + 2.0 * t2 - tau);
    w[1] = 0.5 * (3.0 * t3 - 5.0 * t2 + 2.0);
    w[2] = 0.5 * (-3.0 * t3 + 4.0 * t2 + tau);
    w[3] = 0.5 * (t3 - t2);
    d[0] = 0.5 * (-3.0 * t2 + 4.0 * tau - 1.0) * inv_dp;
    d[1] = 0.5 * (9.0 * t2 - 10.0 * tau) * inv_dp;
    d[2] = 0.5 * (-9.0 * t2 + 8.0 * tau + 1.0) * inv_dp;
    d[3] = 0.5 * (3.0 * t2 - 2.0 * tau) * inv_dp;
}

// Colour-law evaluation modes of one evaluation (decided in the prologue, warp-uniform):
//   CM_GENERIC  clamp + polynomial + linear continuation (any sample anywhere)
//   CM_INSIDE   every in-range sample lies inside [cl_lo, cl_hi]: polynomial only
//   CM_LINEAR   every sample lies on one side outside the range: CL = lin_a + lin_b * dlam
enum { CM_GENERIC = 0, CM_INSIDE = 1, CM_LINEAR = 2 };

// ---- shared-memory records -----------------------------------------------------------------
// Per unit (supernova x sample) of the current group.
template <typename T> struct UnitRec {
    T cl[SB_MAX_CL];      // colour-law coefficients (fp32 forward mode: times c*log2e)
    T s_lo, s_hi;         // continuation slopes (same scaling)
    T al;                 // reduced wavelength per observer-frame Angstrom: r_j = dlam_j*al + be
    T c_exp;              // gradient mode: exponent argument = CL * c_exp
    T x1, a_t;            // a_t: model cells per observer-frame Angstrom
    double x0, opz, t0, cc;
    long long out_base;   // first element of this unit in out_flux
    int32_t sn, o_lo, n_obs, e_begin;
};

// Per evaluation of the current chunk; written by one thread, read by one warp.
template <typename T> struct EvalRecBase {
    int32_t j_lo, j_hi;   // in-range samples [j_lo, j_hi) (absolute index into the band tables)
    int32_t col0;         // first table column loaded by lane 0 of pass 0 (multiple of 4)
    int32_t n_entries;    // coefficient entries (cells) needed; 0 = nothing to integrate
    int32_t rowoff[4];    // element offset of the four phase rows
    T w0[4], w1[4];       // phase weights on M0 and on M1 (forward mode: w1 already times x1)
    T b_t, be;            // t_j = dlam_j*a_t + b_t ; r_j = dlam_j*al + be
    int32_t unit, obs;    // group-local unit, global observation index
    double scale;         // zero-point factor S
    T lin_a, lin_b;       // CM_LINEAR: CL_j = lin_a + lin_b * dlam_j (scaled like UnitRec::cl)
    int32_t cmode;        // colour-law mode of this evaluation (CM_*)
    int32_t pad_;
};
template <typename T, bool GRAD> struct EvalRec : EvalRecBase<T> {};
template <typename T> struct EvalRec<T, true> : EvalRecBase<T> {
    T d0[4], d1[4];       // d/dp weights on M0 and on M1 (d1 already times x1)
};

template <typename T, bool GRAD> struct SmemLayout {
    // byte offsets of the carve-up; every block is 16-byte aligned
    size_t rowbuf, recs, res, units, uacc, misc, bands, total;
    __host__ __device__ SmemLayout(int nwarps, int tile_cells, int cap, int n_band_total, bool stage)
    {
        constexpr int NSET = GRAD ? 3 : 1;
        constexpr int NRES = GRAD ? 5 : 1;
        size_t o = 0;
        rowbuf = o; o += (size_t)nwarps * tile_cells * NSET * sizeof(typename Vec4<T>::type);
        recs = o; o += (size_t)cap * sizeof(EvalRec<T, GRAD>);
        res = o; o += (size_t)cap * NRES * sizeof(double);
        units = o; o += (size_t)kMaxGroup * sizeof(UnitRec<T>);
        uacc = o; o += (size_t)kMaxGroup * 5 * sizeof(double);
        misc = o; o += 16;
        bands = o; o += stage ? (size_t)((n_band_total + 1) & ~1) * sizeof(typename Vec2<T>::type) : 0;
        total = o;
    }
};

// ---- prologue: one thread per evaluation ----------------------------------------------------
// Fills the evaluation's record, or (nothing to integrate / bad band index) its result directly.
template <typename T, bool GRAD>
__device__ __forceinline__ void eval_prologue(const SbKParams &P, const UnitRec<T> *units, int nu, int e,
                                              EvalRec<T, GRAD> &R, double *res,
                                              const typename Vec2<T>::type *tab)
{
    constexpr int NRES = GRAD ? 5 : 1;
    const SbModelParams &mp = P.mp;
    int gu = 0;
    while (gu + 1 < nu && e >= units[gu + 1].e_begin) ++gu;
    const UnitRec<T> &U = units[gu];
    const int o = U.o_lo + (e - U.e_begin);
    R.unit = gu;
    R.obs = o;
    R.n_entries = 0;
#pragma unroll
    for (int k = 0; k < NRES; ++k) res[k] = 0.0;
    const int b = __ldg(P.band + o);
    if ((unsigned)b >= (unsigned)P.n_bands) {
#pragma unroll
        for (int k = 0; k < NRES; ++k) res[k] = __longlong_as_double(0x7ff8000000000000LL);
        return;
    }
    const int nP = mp.n_phase, nW = mp.n_wave;
    const double inv_dp = 1.0 / mp.dp, inv_dl = 1.0 / mp.dl;
    const int boff = __ldg(P.band_off + b);
    const int nb = __ldg(P.band_off + b + 1) - boff;
    const double lam_first = __ldg(P.band_lam_first + b);
    const double opz = U.opz, inv_opz = 1.0 / opz;
    // ---- a1: phase
    const double p = ((double)static_cast<const T *>(P.time)[o] - U.t0) / opz;
    const double up = (p - mp.p0) * inv_dp;
    if (!((up >= 0.0) && (up <= (double)(nP - 1)))) return;
    // in-range band samples [j_lo, j_hi): 0 <= u_j <= nW-1; membership is decided in fp64
    // (dlam_j is exact for fp32-representable grids)
    const double dl_lo = mp.l0 * opz - lam_first;
    const double dl_hi = (mp.l0 + (double)(nW - 1) * mp.dl) * opz - lam_first;
    auto probe = [&](int j) { return (double)tab[boff + j].x; };
    const int j_lo = count_less(nb, dl_lo, probe, false);
    const int j_hi = count_less(nb, dl_hi, probe, true);
    if (j_lo >= j_hi) return;
    // ---- a2: phase weights
    const int kp = min((int)floor(up), nP - 2);
    const double tau = up - (double)kp;
    const bool pborder = (kp == 0) || (kp == nP - 2);
    double wv[4], wd[4];
    phase_weights(tau, pborder, inv_dp, wv, wd);
    const double x1 = (double)U.x1;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        R.rowoff[k] = min(max(kp - 1 + k, 0), nP - 1) * mp.ld;
        R.w0[k] = (T)wv[k];
        R.w1[k] = GRAD ? (T)wv[k] : (T)(wv[k] * x1);
        if constexpr (GRAD) {
            R.d0[k] = (T)wd[k];
            R.d1[k] = (T)(wd[k] * x1);
        }
    }
    // ---- a1: wavelength geometry relative to the first cell of the window
    const double a_d = inv_opz * inv_dl;                          // cells per observer-frame Angstrom
    const double ub = (lam_first * inv_opz - mp.l0) * inv_dl;     // u of dlam = 0
    const double u_first = (double)tab[boff + j_lo].x * a_d + ub;
    const double u_last = (double)tab[boff + j_hi - 1].x * a_d + ub;
    const int i_first = min(max((int)floor(u_first), 0), nW - 2);
    const int i_last = min(max((int)floor(u_last), 0), nW - 2);
    // window of cells i_first-1 .. i_last+1 (one spare cell each side for fp32 rounding of t_j);
    // entry q <-> cell g0 + q, g0 aligned so that table columns are loaded as aligned float4
    const int col0 = ((i_first - 1 + SB_PAD_L) & ~3) - 4;
    const int g0 = col0 + 4 - SB_PAD_L;
    R.col0 = col0;
    R.n_entries = i_last + 1 - g0 + 1;
    R.j_lo = boff + j_lo;
    R.j_hi = boff + j_hi;
    R.b_t = (T)(ub - (double)g0 - 0.5); // t_j = u_j - g0 - 1/2, rint(t_j) = entry, remainder in [-1/2, 1/2]
    const double al_d = inv_opz * mp.cl_inv_span;
    const double be_d = (lam_first * inv_opz - mp.cl_b) * mp.cl_inv_span;
    R.be = (T)be_d;
    // ---- a3: colour-law mode of this evaluation (reduced wavelength is monotone in j)
    {
        const double r_a = (double)tab[boff + j_lo].x * al_d + be_d;
        const double r_b = (double)tab[boff + j_hi - 1].x * al_d + be_d;
        const double r_min = fmin(r_a, r_b), r_max = fmax(r_a, r_b);
        const double margin = 1e-4; // far above the fp32 rounding of r_j, so every lane agrees with the mode
        const double cscale = GRAD ? 1.0 : U.cc * exp_arg_scale<T>();
        int cmode = CM_GENERIC;
        double lin_a = 0.0, lin_b = 0.0;
        if (r_min >= mp.r_lo + margin && r_max <= mp.r_hi - margin) {
            cmode = CM_INSIDE;
        } else if (r_min >= mp.r_hi + margin) {
            cmode = CM_LINEAR;
            lin_a = (mp.p_hi + mp.s_hi * (be_d - mp.r_hi)) * cscale;
            lin_b = mp.s_hi * al_d * cscale;
        } else if (r_max <= mp.r_lo - margin) {
            cmode = CM_LINEAR;
            lin_a = (mp.p_lo + mp.s_lo * (be_d - mp.r_lo)) * cscale;
            lin_b = mp.s_lo * al_d * cscale;
        }
        R.cmode = cmode;
        R.lin_a = (T)lin_a;
        R.lin_b = (T)lin_b;
    }
    double S = 1.0;
    if (P.zp != nullptr) S = exp10(0.4 * (double)static_cast<const T *>(P.zp)[o]) * __ldg(P.band_zpab_inv + b);
    R.scale = S;
}

// ---- shared-memory access through 32-bit addresses (no generic-pointer arithmetic in the loops)
__device__ __forceinline__ uint32_t smem_addr(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void sts_v4(uint32_t a, const float4 &v)
{
    asm volatile("st.shared.v4.f32 [%0], {%1, %2, %3, %4};" ::"r"(a), "f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w) : "memory");
}
__device__ __forceinline__ void sts_v4(uint32_t a, const double4 &v)
{
    asm volatile("st.shared.v2.f64 [%0], {%1, %2};" ::"r"(a), "d"(v.x), "d"(v.y) : "memory");
    asm volatile("st.shared.v2.f64 [%0+16], {%1, %2};" ::"r"(a), "d"(v.z), "d"(v.w) : "memory");
}
__device__ __forceinline__ void lds_v4(uint32_t a, float4 &v)
{
    asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(a));
}
__device__ __forceinline__ void lds_v4(uint32_t a, double4 &v)
{
    asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(a));
    asm volatile("ld.shared.v2.f64 {%0, %1}, [%2+16];" : "=d"(v.z), "=d"(v.w) : "r"(a));
}

// Split t into a row-buffer key and the signed remainder s = t - rint(t), |s| <= 1/2.
//   fp32: magic-number rounding on the FMA pipe (no F2I/FRND on the quarter-rate XU pipe); the key
//   is the raw bit pattern of t + 1.5*2^23, i.e. rint(t) + kKeyBias<float>.   fp64: key = rint(t).
// The slot of entry q is swz(q); since the bias and the tile origin are multiples of 32, swz(key)
// = swz(q) + bias, and the bias is folded into the base address once per tile.
template <typename T> struct KeyBias;
template <> struct KeyBias<float> { static constexpr uint32_t value = 0x4B400000u; };
template <> struct KeyBias<double> { static constexpr uint32_t value = 0u; };
__device__ __forceinline__ void split_key(float t, uint32_t &key, float &s)
{
    const float magic = 12582912.0f; // 1.5 * 2^23: valid for |t| < 2^22
    const float r = __fadd_rn(t, magic);
    key = __float_as_uint(r);
    s = __fsub_rn(t, __fsub_rn(r, magic));
}
__device__ __forceinline__ void split_key(double t, uint32_t &key, double &s)
{
    const int i = __double2int_rn(t);
    key = (uint32_t)i;
    s = t - (double)i;
}
__device__ __forceinline__ uint32_t swz_key(uint32_t k) { return k ^ ((k >> 3) & 3u); }

template <typename T, int NCL> struct Colour {
    T a[NCL];        // polynomial coefficients
    T r_lo, r_hi;    // clamp range of the reduced wavelength
    T s_lo, s_hi;    // continuation slopes (same scaling as a[])
    T al, be;        // r_j = dlam_j * al + be
    T lin_a, lin_b;  // CM_LINEAR
    template <int CM> __device__ __forceinline__ T eval(T dl) const
    {
        if constexpr (CM == CM_LINEAR) {
            return fma_t(dl, lin_b, lin_a);
        } else if constexpr (CM == CM_INSIDE) {
            const T r = fma_t(dl, al, be);
            T p = a[NCL - 1];
#pragma unroll
            for (int q = NCL - 2; q >= 0; --q) p = fma_t(p, r, a[q]);
            return p;
        } else {
            const T r = fma_t(dl, al, be);
            const T rc = fmin(fmax(r, r_lo), r_hi);
            const T d = r - rc;
            const T slope = d > (T)0 ? s_hi : s_lo;
            T p = a[NCL - 1];
#pragma unroll
            for (int q = NCL - 2; q >= 0; --q) p = fma_t(p, rc, a[q]);
            return fma_t(slope, d, p);
        }
    }
};

// ---- main: one warp integrates one evaluation -------------------------------------------------
constexpr int kPassesPerTile = 3; // a tile is at most 3 collapse passes (360 entries)

template <typename T, bool GRAD, int NCL>
__device__ __forceinline__ void eval_warp(const SbKParams &P, const UnitRec<T> &U, const EvalRec<T, GRAD> &R,
                                          uint32_t rowbuf_s, int TC,
                                          const typename Vec2<T>::type *__restrict__ tab, int lane, double *res)
{
    using V4 = typename Vec4<T>::type;
    using V2 = typename Vec2<T>::type;
    constexpr int NSET = GRAD ? 3 : 1;
    constexpr uint32_t kSlot = (uint32_t)sizeof(V4) * NSET; // bytes per row-buffer entry
    const SbModelParams &mp = P.mp;
    const int nW = mp.n_wave;
    const T *__restrict__ M0 = static_cast<const T *>(P.m0);
    const T *__restrict__ M1 = static_cast<const T *>(P.m1);

    const int n_entries = R.n_entries, col0 = R.col0, j_hi = R.j_hi;
    const int g0 = col0 + 4 - SB_PAD_L;
    const int col_max = col0 + 4 + n_entries + 1; // last node column any needed cell touches
    T w0[4], w1[4], d0[4], d1[4];
    const T *p0[4], *p1[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        w0[k] = R.w0[k];
        w1[k] = R.w1[k];
        if constexpr (GRAD) { d0[k] = R.d0[k]; d1[k] = R.d1[k]; }
        p0[k] = M0 + (R.rowoff[k] + col0 + 4 * lane);
        p1[k] = M1 + (R.rowoff[k] + col0 + 4 * lane);
    }
    const T x1_t = U.x1;
    const T a_t = U.a_t, b_t = R.b_t;
    Colour<T, NCL> col;
#pragma unroll
    for (int q = 0; q < NCL; ++q) col.a[q] = U.cl[q];
    col.r_lo = (T)mp.r_lo;
    col.r_hi = (T)mp.r_hi;
    col.s_lo = U.s_lo;
    col.s_hi = U.s_hi;
    col.al = U.al;
    col.be = R.be;
    col.lin_a = R.lin_a;
    col.lin_b = R.lin_b;
    const T c_exp = U.c_exp;
    const int cmode = R.cmode;

    T accF = 0, accB = 0, accC = 0, accD = 0;
    int ja = R.j_lo;
    const int tile_step = (TC - 8) & ~31; // tile origins stay multiples of 32 (see split_key)
    for (int q0 = 0;; q0 += tile_step) {
        const int q_end = min(q0 + TC, n_entries);
        // ---- a2: collapse the phase rows (4 nodes per lane), convert to per-cell cubic coefficients
#pragma unroll
        for (int ps = 0; ps < kPassesPerTile; ++ps) {
            const int qp = q0 + ps * kCellsPerPass;
            if (qp >= q_end) break;
            const int c = col0 + qp + 4 * lane; // this lane's nodes: columns c..c+3 = cells' left nodes
            T r[4] = {0, 0, 0, 0}, r1[4] = {0, 0, 0, 0}, rd[4] = {0, 0, 0, 0};
            if (c <= col_max) {
                V4 v0[4], v1[4];
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    v0[k] = ldg_v4(p0[k] + ps * kCellsPerPass);
                    v1[k] = ldg_v4(p1[k] + ps * kCellsPerPass);
                }
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    const T a0[4] = {v0[k].x, v0[k].y, v0[k].z, v0[k].w};
                    const T a1[4] = {v1[k].x, v1[k].y, v1[k].z, v1[k].w};
#pragma unroll
                    for (int e = 0; e < 4; ++e) {
                        r[e] = fma_t(w0[k], a0[e], r[e]);
                        if constexpr (GRAD) {
                            r1[e] = fma_t(w1[k], a1[e], r1[e]);
                            rd[e] = fma_t(d0[k], a0[e], rd[e]);
                            rd[e] = fma_t(d1[k], a1[e], rd[e]);
                        } else {
                            r[e] = fma_t(w1[k], a1[e], r[e]);
                        }
                    }
                }
                if constexpr (GRAD) {
#pragma unroll
                    for (int e = 0; e < 4; ++e) r[e] = fma_t(x1_t, r1[e], r[e]);
                }
            }
            const int qb = qp + 4 * (lane - 1);       // first entry this lane produces (lanes 1..30)
            const int gb = g0 + qb;                   // its cell index
            const bool special = (g0 + qp <= 0) || (g0 + qp + kCellsPerPass + 3 >= nW - 2); // warp-uniform
            const bool writer = (lane >= 1) && (lane <= 30);
            // lane l's four entries live in one 8-slot swizzle group half: slots (qb-q0)+e ^ x, x fixed
            const uint32_t qrel = (uint32_t)(qb - q0);
            const uint32_t x = (qrel >> 3) & 3u;
            auto emit = [&](const T(&n4)[4], int set) {
                const T am = __shfl_up_sync(0xffffffffu, n4[3], 1);
                const T ap = __shfl_down_sync(0xffffffffu, n4[0], 1);
                const T ap2 = __shfl_down_sync(0xffffffffu, n4[1], 1);
                const T n[7] = {am, n4[0], n4[1], n4[2], n4[3], ap, ap2};
                V4 cf[4];
                if (!special) {
#pragma unroll
                    for (int e = 0; e < 4; ++e) cf[e] = cell_coef_interior<T>(n[e], n[e + 1], n[e + 2], n[e + 3]);
                } else {
#pragma unroll
                    for (int e = 0; e < 4; ++e) cf[e] = cell_coef<T>(gb + e, nW, n[e], n[e + 1], n[e + 2], n[e + 3]);
                }
                if (writer) {
#pragma unroll
                    for (int e = 0; e < 4; ++e)
                        if (qb + e < q_end) sts_v4(rowbuf_s + ((qrel + e) ^ x) * kSlot + set * (uint32_t)sizeof(V4), cf[e]);
                }
            };
            emit(r, 0);
            if constexpr (GRAD) {
                emit(r1, 1);
                emit(rd, 2);
            }
        }
        __syncwarp();
        // ---- samples of this tile: rint(t_j) in [q0, q0+TC-2]
        int jb = j_hi;
        if (q_end < n_entries) {
            const T thr = (T)(q0 + TC) - (T)1.5;
            auto probe = [&](int j) { return fma_t(tab[ja + j].x, a_t, b_t); };
            jb = ja + warp_count_less(j_hi - ja, thr, lane, probe);
        }
        const uint32_t base = rowbuf_s - (KeyBias<T>::value + (uint32_t)q0) * kSlot;
        auto samples = [&](auto cm_tag) {
            constexpr int CM = decltype(cm_tag)::value;
#pragma unroll 4
            for (int j = ja + lane; j < jb; j += kWarpSize) {
                const V2 dw = tab[j];
                const T dl = dw.x, wj = dw.y;
                uint32_t key;
                T s;
                split_key(fma_t(dl, a_t, b_t), key, s);
                const uint32_t addr = swz_key(key) * kSlot + base;
                V4 cf;
                lds_v4(addr, cf);
                const T val = poly3<T>(cf, s);
                const T cl = col.template eval<CM>(dl);
                if constexpr (GRAD) {
                    V4 c1, cd;
                    lds_v4(addr + (uint32_t)sizeof(V4), c1);
                    lds_v4(addr + 2u * (uint32_t)sizeof(V4), cd);
                    const T ew = exp_scaled(cl * c_exp) * wj;
                    const T v1 = poly3<T>(c1, s);
                    const T vd = poly3<T>(cd, s);
                    const T f = ew * val;
                    accF += f;
                    accB = fma_t(ew, v1, accB);
                    accC = fma_t(f, cl, accC);
                    accD = fma_t(ew, vd, accD);
                } else {
                    accF = fma_t(exp_scaled(cl) * wj, val, accF);
                }
            }
        };
        if (cmode == CM_INSIDE) samples(std::integral_constant<int, CM_INSIDE>{});
        else if (cmode == CM_LINEAR) samples(std::integral_constant<int, CM_LINEAR>{});
        else samples(std::integral_constant<int, CM_GENERIC>{});
        ja = jb;
        __syncwarp();
        if (q_end >= n_entries) break;
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            p0[k] += tile_step;
            p1[k] += tile_step;
        }
    }
    // ---- a5: wavelength integral (warp butterfly), a6: zero point
    accF = warp_sum(accF);
    if constexpr (GRAD) {
        accB = warp_sum(accB);
        accC = warp_sum(accC);
        accD = warp_sum(accD);
    }
    if (lane == 0) {
        const double S = R.scale, x0 = U.x0;
        res[0] = S * x0 * (double)accF;
        if constexpr (GRAD) {
            res[1] = S * (double)accF;
            res[2] = S * x0 * (double)accB;
            res[3] = S * x0 * (double)accC;
            res[4] = -S * x0 * (double)accD / U.opz;
        }
    }
}

// ---- the kernel -------------------------------------------------------------------------------
template <typename T, bool GRAD, int NCL, bool STAGE, int NWARPS>
__global__ void __launch_bounds__(NWARPS * kWarpSize, 1) sb_fused_kernel(const __grid_constant__ SbKParams P)
{
    using V4 = typename Vec4<T>::type;
    using V2 = typename Vec2<T>::type;
    constexpr int NSET = GRAD ? 3 : 1; // coefficient sets per cell: value [, M1-only, d/dphase]
    constexpr int NRES = GRAD ? 5 : 1; // results per evaluation: m [, dm/d(x0, x1, c, t0)]
    constexpr int NT = NWARPS * kWarpSize;
    extern __shared__ __align__(16) unsigned char smem_raw[];

    if (P.n_live != nullptr && __ldg(P.n_live) == 0) return; // fit driver: every lane has stopped
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const SbModelParams &mp = P.mp;
    const int TC = P.tile_cells, CAP = P.chunk_cap, G = P.group_units;
    const SmemLayout<T, GRAD> L(NWARPS, TC, CAP, P.n_band_total, STAGE);
    const uint32_t rowbuf_s = smem_addr(smem_raw + L.rowbuf) + (uint32_t)warp * (uint32_t)TC * (uint32_t)(NSET * sizeof(V4));
    EvalRec<T, GRAD> *recs = reinterpret_cast<EvalRec<T, GRAD> *>(smem_raw + L.recs);
    double *res = reinterpret_cast<double *>(smem_raw + L.res);
    UnitRec<T> *units = reinterpret_cast<UnitRec<T> *>(smem_raw + L.units);
    double *uacc = reinterpret_cast<double *>(smem_raw + L.uacc);
    int *misc = reinterpret_cast<int *>(smem_raw + L.misc); // [0] work counter, [1] evaluations in the group
    const V2 *tab = static_cast<const V2 *>(P.band_tab);
    if (STAGE) {
        V2 *s_tab = reinterpret_cast<V2 *>(smem_raw + L.bands);
        for (int i = tid; i < P.n_band_total; i += NT) s_tab[i] = tab[i];
        tab = s_tab;
        __syncthreads();
    }
    T *o_flux = static_cast<T *>(P.out_flux);
    T *o_dflux = static_cast<T *>(P.out_dflux);
    const T *__restrict__ g_flux = static_cast<const T *>(P.flux);
    const T *__restrict__ g_err = static_cast<const T *>(P.fluxerr);
    const bool want_chi = (P.out_chi2 != nullptr) || (P.out_dchi2 != nullptr);
    const long long n_units = (long long)P.n_sn * P.n_samples;
    const long long n_groups = (n_units + G - 1) / G;

    for (long long group = blockIdx.x; group < n_groups; group += gridDim.x) {
        const long long u0 = group * G;
        const int nu = (int)min((long long)G, n_units - u0);
        // ---- unit records (one thread per unit)
        if (tid < nu) {
            const long long unit = u0 + tid;
            UnitRec<T> &U = units[tid];
            const int sn = (int)(unit / P.n_samples);
            const int ks = (int)(unit - (long long)sn * P.n_samples);
            const int o_lo = __ldg(P.obs_offset + sn);
            const int n_obs = __ldg(P.obs_offset + sn + 1) - o_lo;
            const double z = (double)static_cast<const T *>(P.z)[sn];
            const double cc = (double)static_cast<const T *>(P.c)[unit];
            const double opz = 1.0 + z, inv_opz = 1.0 / opz;
            U.sn = sn;
            U.o_lo = o_lo;
            U.n_obs = n_obs;
            U.out_base = (long long)o_lo * P.n_samples + (long long)ks * n_obs;
            U.x0 = (double)static_cast<const T *>(P.x0)[unit];
            U.x1 = static_cast<const T *>(P.x1)[unit];
            U.t0 = (double)static_cast<const T *>(P.t0)[unit];
            U.cc = cc;
            U.opz = opz;
            U.a_t = (T)(inv_opz / mp.dl);
            U.al = (T)(inv_opz * mp.cl_inv_span);
            // colour law of this unit (a3).  Forward fp32: fold c*log2e into the coefficients.
            const double cscale = GRAD ? 1.0 : cc * exp_arg_scale<T>();
#pragma unroll
            for (int q = 0; q < SB_MAX_CL; ++q) U.cl[q] = (T)(mp.cl[q] * cscale);
            U.s_lo = (T)(mp.s_lo * cscale);
            U.s_hi = (T)(mp.s_hi * cscale);
            U.c_exp = (T)(cc * exp_arg_scale<T>());
        }
        if (tid < kMaxGroup * 5) uacc[tid] = 0.0;
        __syncthreads();
        if (tid == 0) {
            int acc = 0;
            for (int u = 0; u < nu; ++u) {
                units[u].e_begin = acc;
                acc += units[u].n_obs;
            }
            misc[1] = acc;
        }
        __syncthreads();
        const int n_ev = misc[1];

        for (int c0 = 0; c0 < n_ev; c0 += CAP) {
            const int nc = min(CAP, n_ev - c0);
            // ---- prologue: one thread per evaluation
            for (int el = tid; el < nc; el += NT)
                eval_prologue<T, GRAD>(P, units, nu, c0 + el, recs[el], res + (size_t)el * NRES, tab);
            if (tid == 0) misc[0] = 0;
            __syncthreads();
            // ---- main: warps pull evaluations
            for (;;) {
                int el = 0;
                if (lane == 0) el = atomicAdd(&misc[0], 1);
                el = __shfl_sync(0xffffffffu, el, 0);
                if (el >= nc) break;
                const EvalRec<T, GRAD> &R = recs[el];
                if (R.n_entries > 0)
                    eval_warp<T, GRAD, NCL>(P, units[R.unit], R, rowbuf_s, TC, tab, lane, res + (size_t)el * NRES);
            }
            __syncthreads();
            // ---- epilogue: results out (coalesced within a unit), chi^2 terms in place (a7)
            for (int el = tid; el < nc; el += NT) {
                const EvalRec<T, GRAD> &R = recs[el];
                const UnitRec<T> &U = units[R.unit];
                double *rr = res + (size_t)el * NRES;
                const long long oi = U.out_base + (R.obs - U.o_lo);
                const double m = rr[0];
                if (o_flux) o_flux[oi] = (T)m;
                if constexpr (GRAD) {
                    if (o_dflux) reinterpret_cast<V4 *>(o_dflux)[oi] = make_v4<T>((T)rr[1], (T)rr[2], (T)rr[3], (T)rr[4]);
                }
                if (want_chi) {
                    const double f = (double)g_flux[R.obs], e = (double)g_err[R.obs];
                    const double q = (f - m) / e;
                    rr[0] = q * q;
                    if constexpr (GRAD) {
                        const double g = -2.0 * (f - m) / (e * e);
                        rr[1] *= g;
                        rr[2] *= g;
                        rr[3] *= g;
                        rr[4] *= g;
                    }
                }
            }
            __syncthreads();
            if (want_chi) { // one warp per unit, lanes stride its terms, fixed butterfly: deterministic
                for (int u = warp; u < nu; u += NWARPS) {
                    const int lo = max(units[u].e_begin, c0) - c0;
                    const int hi = min(units[u].e_begin + units[u].n_obs, c0 + nc) - c0;
                    double s[NRES];
#pragma unroll
                    for (int k = 0; k < NRES; ++k) s[k] = 0.0;
                    for (int el = lo + lane; el < hi; el += kWarpSize) {
#pragma unroll
                        for (int k = 0; k < NRES; ++k) s[k] += res[(size_t)el * NRES + k];
                    }
#pragma unroll
                    for (int k = 0; k < NRES; ++k) s[k] = warp_sum(s[k]);
                    if (lane == 0) {
#pragma unroll
                        for (int k = 0; k < NRES; ++k) uacc[u * 5 + k] += s[k];
                    }
                }
                __syncthreads();
            }
        }
        if (want_chi && tid < nu) {
            const long long unit = u0 + tid;
            if (P.out_chi2) static_cast<T *>(P.out_chi2)[unit] = (T)uacc[tid * 5];
            if constexpr (GRAD) {
                if (P.out_dchi2)
                    reinterpret_cast<V4 *>(P.out_dchi2)[unit] =
                        make_v4<T>((T)uacc[tid * 5 + 1], (T)uacc[tid * 5 + 2], (T)uacc[tid * 5 + 3], (T)uacc[tid * 5 + 4]);
            }
        }
        __syncthreads();
    }
}

} // namespace sb
