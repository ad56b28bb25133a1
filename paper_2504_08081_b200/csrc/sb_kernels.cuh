// sb_kernels.cuh -- the fused SALT3 band-flux kernel (sm_100a).
//
// One CTA per unit (supernova s, parameter sample k), persistent over units; one warp per
// evaluation (observation i of that unit); lanes stride the band's wavelength samples.
// Steps (citations in include/saltband.h):
//   a1  p = (t - t0)/(1+z) per evaluation (fp64 scalar prologue); per sample the fractional cell
//       coordinate u_j = (lam_j/(1+z) - L0)/dL, computed RELATIVE to the evaluation's first cell as
//       one FFMA  t_j = dlam_j * a + b  (dlam_j = lam_j - lam_first is exact in fp32).
//   a2  bicubic interpolation, separable: the <= 4 phase rows of M0 and M1 are collapsed once per
//       evaluation into a 1-D row R[l] = sum_k wp_k (M0 + x1 M1)[kp+k][l]; each cell of that row
//       is then converted to the cubic's coefficients about the cell centre (an exact
//       re-association of the Keys a=-1/2 / Catmull-Rom weights; linear in border cells), stored
//       as one float4 per cell in this warp's shared-memory row buffer.  A sample is 1 LDS.128 +
//       3 FFMA.
//   a3  colour law: degree-(NCL-1) Horner in the reduced wavelength, linear continuation by
//       clamping, one ex2 per sample (coefficients pre-scaled by c*log2(e) in fp32 mode).
//   a4/a5  folded weight W_j = w_j T_j lam_j/(hc) (trapezoid weight folded at load), FFMA
//       accumulate per lane, warp-shuffle butterfly.
//   a6  zero point S = 10^(0.4 zp)/ZPAB_b in fp64 per evaluation.
//   a7  chi^2 per unit: per-warp partial sums in observation order, fixed-order CTA sum (fp64
//       accumulators; deterministic).
//   a8  analytic gradient: three coefficient sets (value row, M1-only row, d/dphase row) and four
//       accumulators give d m/d(x0, x1, c, t0).
#pragma once
#include "sb_internal.h"

namespace sb {

constexpr int kWarpSize = 32;
constexpr int kCellsPerPass = 29; // a 32-node pass yields 29 cells (3-node halo via shuffles)

template <typename T> struct Vec4;
template <> struct Vec4<float> { using type = float4; };
template <> struct Vec4<double> { using type = double4; };

template <typename T> __device__ __forceinline__ typename Vec4<T>::type make_v4(T a, T b, T c, T d);
template <> __device__ __forceinline__ float4 make_v4<float>(float a, float b, float c, float d) { return make_float4(a, b, c, d); }
template <> __device__ __forceinline__ double4 make_v4<double>(double a, double b, double c, double d) { return make_double4(a, b, c, d); }

// Split t into the nearest integer and the signed remainder s = t - rint(t), |s| <= 1/2.
// fp32: magic-number rounding on the FMA pipe (no F2I/FRND on the quarter-rate XU pipe).
__device__ __forceinline__ void split_rn(float t, int &idx, float &s)
{
    const float magic = 12582912.0f; // 1.5 * 2^23: valid for |t| < 2^22
    float r = __fadd_rn(t, magic);
    idx = __float_as_int(r) - 0x4B400000;
    s = __fsub_rn(t, __fsub_rn(r, magic));
}
__device__ __forceinline__ void split_rn(double t, int &idx, double &s)
{
    idx = __double2int_rn(t);
    s = t - (double)idx;
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

// Number of j in [0, n) with f(j) < thr for a non-decreasing f; warp-cooperative 32-ary search.
template <typename F, typename T>
__device__ __forceinline__ int warp_count_less(int n, T thr, int lane, F f, bool or_equal)
{
    int lo = 0, len = n;
    while (len > 0) {
        int step = (len + kWarpSize - 1) / kWarpSize;
        int j = lo + lane * step; // probe the first element of each of 32 sub-ranges
        bool less = false;
        if (j < lo + len) {
            T v = f(j);
            less = or_equal ? (v <= thr) : (v < thr);
        }
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

// Coefficients of one cell's polynomial about the cell centre, s in [-1/2, 1/2].
//   g = global cell index, nodes rm = R[g-1], r0 = R[g], r1 = R[g+1], r2 = R[g+2] (clamped loads).
//   Interior (1 <= g <= n-3): Catmull-Rom.  g = 0 or n-2: linear (G2).  g = -1 and
//   g = n-1 continue the adjacent border line (reached only within rounding of the grid edge).
template <typename T>
__device__ __forceinline__ typename Vec4<T>::type cell_coef(int g, int n, T rm, T r0, T r1, T r2)
{
    const T h = (T)0.5;
    if (g < -1 || g > n - 1) return make_v4<T>(0, 0, 0, 0);
    if (g == -1) { T d = r2 - r1; return make_v4<T>(r1 - h * d, d, 0, 0); }
    if (g == n - 1) { T d = r0 - rm; return make_v4<T>(r0 + h * d, d, 0, 0); }
    if (g == 0 || g == n - 2) return make_v4<T>(h * (r0 + r1), r1 - r0, 0, 0);
    T s1 = r0 + r1, s2 = rm + r2, d1 = r1 - r0, d2 = r2 - rm;
    return make_v4<T>(((T)9 * s1 - s2) * (T)0.0625, ((T)11 * d1 - d2) * (T)0.125, (s2 - s1) * (T)0.25,
                      (d2 - (T)3 * d1) * h);
}

template <typename T>
__device__ __forceinline__ T poly3(const typename Vec4<T>::type &a, T s)
{
    return fma_t(fma_t(fma_t(a.w, s, a.z), s, a.y), s, a.x);
}

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

template <typename T, int NCL> struct Colour {
    T a[NCL];        // polynomial coefficients (fp32 fwd mode: times c*log2e)
    T r_lo, r_hi;    // clamp range of the reduced wavelength
    T s_lo, s_hi;    // continuation slopes (same scaling as a[])
    T al, be;        // r_j = dlam_j * al + be
    // returns CL(r) in the scaling of a[]
    __device__ __forceinline__ T eval(T dl) const
    {
        T r = fma_t(dl, al, be);
        T rc = fmin(fmax(r, r_lo), r_hi);
        T d = r - rc;
        T slope = d > (T)0 ? s_hi : s_lo;
        T p = a[NCL - 1];
#pragma unroll
        for (int q = NCL - 2; q >= 0; --q) p = fma_t(p, rc, a[q]);
        return fma_t(slope, d, p);
    }
};

template <typename T, bool GRAD, int NCL, bool STAGE, int NWARPS>
__global__ void __launch_bounds__(NWARPS * kWarpSize, 1) sb_fused_kernel(const __grid_constant__ SbKParams P)
{
    using V4 = typename Vec4<T>::type;
    constexpr int NSET = GRAD ? 3 : 1; // coefficient sets per cell: value [, M1-only, d/dphase]
    extern __shared__ __align__(16) unsigned char smem_raw[];

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const SbModelParams &mp = P.mp;
    const int TC = P.tile_cells;

    // ---- shared memory carve-up: [warp row buffers][reduction scratch][band tables]
    V4 *rowbuf = reinterpret_cast<V4 *>(smem_raw) + (size_t)warp * TC * NSET;
    double *red = reinterpret_cast<double *>(smem_raw + (size_t)NWARPS * TC * NSET * sizeof(V4));
    const T *tab_dlam = static_cast<const T *>(P.band_dlam);
    const T *tab_w = static_cast<const T *>(P.band_w);
    if (STAGE) {
        T *s_dlam = reinterpret_cast<T *>(red + NWARPS * 5);
        T *s_w = s_dlam + ((P.n_band_total + 3) & ~3);
        for (int i = tid; i < P.n_band_total; i += NWARPS * kWarpSize) {
            s_dlam[i] = tab_dlam[i];
            s_w[i] = tab_w[i];
        }
        tab_dlam = s_dlam;
        tab_w = s_w;
        __syncthreads();
    }
    const T *__restrict__ M0 = static_cast<const T *>(P.m0);
    const T *__restrict__ M1 = static_cast<const T *>(P.m1);
    const T *__restrict__ g_time = static_cast<const T *>(P.time);
    const T *__restrict__ g_zp = static_cast<const T *>(P.zp);
    const T *__restrict__ g_flux = static_cast<const T *>(P.flux);
    const T *__restrict__ g_err = static_cast<const T *>(P.fluxerr);
    T *o_flux = static_cast<T *>(P.out_flux);
    T *o_dflux = static_cast<T *>(P.out_dflux);
    const bool want_chi = (P.out_chi2 != nullptr) || (P.out_dchi2 != nullptr);

    const int nP = mp.n_phase, nW = mp.n_wave, ld = mp.ld;
    const double inv_dp = 1.0 / mp.dp, inv_dl = 1.0 / mp.dl;
    const long long n_units = (long long)P.n_sn * P.n_samples;

    for (long long unit = blockIdx.x; unit < n_units; unit += gridDim.x) {
        const int sn = (int)(unit / P.n_samples);
        const int ks = (int)(unit - (long long)sn * P.n_samples);
        const int o_lo = __ldg(P.obs_offset + sn);
        const int n_obs = __ldg(P.obs_offset + sn + 1) - o_lo;
        const double z = (double)static_cast<const T *>(P.z)[sn];
        const double x0 = (double)static_cast<const T *>(P.x0)[unit];
        const double x1 = (double)static_cast<const T *>(P.x1)[unit];
        const double cc = (double)static_cast<const T *>(P.c)[unit];
        const double t0 = (double)static_cast<const T *>(P.t0)[unit];
        const double opz = 1.0 + z;
        const double inv_opz = 1.0 / opz;
        const double a_d = inv_opz * inv_dl; // cells per observer-frame Angstrom
        const T a_t = (T)a_d;

        // colour law for this unit (a3).  Forward fp32: fold c*log2e into the coefficients.
        Colour<T, NCL> col;
        const double cscale = GRAD ? 1.0 : cc * exp_arg_scale<T>();
#pragma unroll
        for (int q = 0; q < NCL; ++q) col.a[q] = (T)(mp.cl[q] * cscale);
        col.r_lo = (T)mp.r_lo;
        col.r_hi = (T)mp.r_hi;
        col.s_lo = (T)(mp.s_lo * cscale);
        col.s_hi = (T)(mp.s_hi * cscale);
        const double al_d = inv_opz * mp.cl_inv_span;
        col.al = (T)al_d;
        const T c_exp = (T)(cc * exp_arg_scale<T>()); // GRAD: arg = CL * c_exp

        const long long out_base = (long long)o_lo * P.n_samples + (long long)ks * n_obs;
        double chi = 0.0, dchi0 = 0.0, dchi1 = 0.0, dchi2 = 0.0, dchi3 = 0.0;

        for (int i = warp; i < n_obs; i += NWARPS) {
            const int o = o_lo + i;
            const int b = __ldg(P.band + o);
            double m = 0.0, dm0 = 0.0, dm1 = 0.0, dm2 = 0.0, dm3 = 0.0;
            if ((unsigned)b >= (unsigned)P.n_bands) {
                m = dm0 = dm1 = dm2 = dm3 = __longlong_as_double(0x7ff8000000000000LL);
            } else {
                const int boff = __ldg(P.band_off + b);
                const int nb = __ldg(P.band_off + b + 1) - boff;
                const double lam_first = __ldg(P.band_lam_first + b);
                const T *dlam = tab_dlam + boff;
                const T *wtab = tab_w + boff;
                // ---- a1: phase
                const double p = ((double)g_time[o] - t0) / opz;
                const double up = (p - mp.p0) * inv_dp;
                // in-range band samples [j_lo, j_hi): 0 <= u_j <= nW-1
                const double dl_lo = mp.l0 * opz - lam_first;
                const double dl_hi = (mp.l0 + (double)(nW - 1) * mp.dl) * opz - lam_first;
                int j_lo = 0, j_hi = 0;
                const bool phase_ok = (up >= 0.0) && (up <= (double)(nP - 1));
                if (phase_ok) {
                    // membership is decided in fp64 (dlam_j is exact for fp32-representable grids)
                    auto probe = [&](int j) { return (double)dlam[j]; };
                    j_lo = warp_count_less(nb, dl_lo, lane, probe, false);
                    j_hi = warp_count_less(nb, dl_hi, lane, probe, true);
                }
                if (j_lo < j_hi) {
                    int kp = min((int)floor(up), nP - 2);
                    const double tau = up - (double)kp;
                    const bool pborder = (kp == 0) || (kp == nP - 2);
                    double wv[4], wd[4];
                    phase_weights(tau, pborder, inv_dp, wv, wd);
                    int row[4];
#pragma unroll
                    for (int k = 0; k < 4; ++k) row[k] = min(max(kp - 1 + k, 0), nP - 1) * ld;
                    T w0[4], w1[4], d0[4], d1[4];
#pragma unroll
                    for (int k = 0; k < 4; ++k) {
                        w0[k] = (T)wv[k];
                        w1[k] = GRAD ? (T)wv[k] : (T)(wv[k] * x1);
                        d0[k] = (T)wd[k];
                        d1[k] = (T)(wd[k] * x1);
                    }
                    const T x1_t = (T)x1;
                    // ---- a1: wavelength geometry relative to the first cell
                    const double ub = (lam_first * inv_opz - mp.l0) * inv_dl; // u of dlam = 0
                    const double u_first = (double)dlam[j_lo] * a_d + ub;
                    const double u_last = (double)dlam[j_hi - 1] * a_d + ub;
                    const int i_first = min(max((int)floor(u_first), 0), nW - 2);
                    const int i_last = min(max((int)floor(u_last), 0), nW - 2);
                    const int n_entries = i_last - i_first + 3; // cells i_first-1 .. i_last+1
                    const T b_t = (T)(ub - (double)i_first + 0.5); // t_j = u_j - (i_first-1) - 1/2
                    col.be = (T)((lam_first * inv_opz - mp.cl_b) * mp.cl_inv_span);

                    T accF = 0, accB = 0, accC = 0, accD = 0;
                    int ja = j_lo;
                    for (int q0 = 0; ja < j_hi; q0 += TC - 2) {
                        const int q_end = min(q0 + TC, n_entries);
                        // ---- a2: collapse phase rows, convert to per-cell cubic coefficients
                        for (int qs = q0; qs < q_end; qs += kCellsPerPass) {
                            const int g_lane = i_first - 1 + qs + lane - 1; // lane l: node of cell qs+l-1
                            const int node = min(max(g_lane, 0), nW - 1);
                            T r = 0, r1 = 0, rd = 0;
#pragma unroll
                            for (int k = 0; k < 4; ++k) {
                                const T v0 = __ldg(M0 + row[k] + node);
                                const T v1 = __ldg(M1 + row[k] + node);
                                r = fma_t(w0[k], v0, r);
                                if (GRAD) {
                                    r1 = fma_t(w1[k], v1, r1);
                                    rd = fma_t(d0[k], v0, rd);
                                    rd = fma_t(d1[k], v1, rd);
                                } else {
                                    r = fma_t(w1[k], v1, r);
                                }
                            }
                            if (GRAD) r = fma_t(x1_t, r1, r);
                            const int q = qs + lane - 1; // entry this lane produces (lanes 1..29)
                            {
                                T am = __shfl_up_sync(0xffffffffu, r, 1);
                                T ap = __shfl_down_sync(0xffffffffu, r, 1);
                                T a2 = __shfl_down_sync(0xffffffffu, r, 2);
                                V4 cf = cell_coef<T>(g_lane, nW, am, r, ap, a2);
                                if (lane >= 1 && lane <= kCellsPerPass && q < q_end) rowbuf[(q - q0) * NSET] = cf;
                            }
                            if (GRAD) {
                                T am = __shfl_up_sync(0xffffffffu, r1, 1);
                                T ap = __shfl_down_sync(0xffffffffu, r1, 1);
                                T a2 = __shfl_down_sync(0xffffffffu, r1, 2);
                                V4 cf = cell_coef<T>(g_lane, nW, am, r1, ap, a2);
                                if (lane >= 1 && lane <= kCellsPerPass && q < q_end) rowbuf[(q - q0) * NSET + 1] = cf;
                                am = __shfl_up_sync(0xffffffffu, rd, 1);
                                ap = __shfl_down_sync(0xffffffffu, rd, 1);
                                a2 = __shfl_down_sync(0xffffffffu, rd, 2);
                                cf = cell_coef<T>(g_lane, nW, am, rd, ap, a2);
                                if (lane >= 1 && lane <= kCellsPerPass && q < q_end) rowbuf[(q - q0) * NSET + 2] = cf;
                            }
                        }
                        __syncwarp();
                        // ---- samples of this tile: rint(t_j) in [q0, q0+TC-2]
                        int jb = j_hi;
                        if (q_end < n_entries) {
                            const T thr = (T)(q0 + TC) - (T)1.5;
                            auto probe = [&](int j) { return fma_t(dlam[ja + j], a_t, b_t); };
                            jb = ja + warp_count_less(j_hi - ja, thr, lane, probe, false);
                        }
                        const V4 *rb = rowbuf - (size_t)q0 * NSET;
#pragma unroll 4
                        for (int j = ja + lane; j < jb; j += kWarpSize) {
                            const T dl = dlam[j];
                            const T wj = wtab[j];
                            int idx;
                            T s;
                            split_rn(fma_t(dl, a_t, b_t), idx, s);
                            const V4 cf = rb[idx * NSET];
                            const T val = poly3<T>(cf, s);
                            const T cl = col.eval(dl);
                            if (GRAD) {
                                const T ew = exp_scaled(cl * c_exp) * wj;
                                const T v1 = poly3<T>(rb[idx * NSET + 1], s);
                                const T vd = poly3<T>(rb[idx * NSET + 2], s);
                                const T f = ew * val;
                                accF += f;
                                accB = fma_t(ew, v1, accB);
                                accC = fma_t(f, cl, accC);
                                accD = fma_t(ew, vd, accD);
                            } else {
                                accF = fma_t(exp_scaled(cl) * wj, val, accF);
                            }
                        }
                        ja = jb;
                        __syncwarp();
                        if (q_end >= n_entries) break;
                    }
                    // ---- a5: wavelength integral (warp butterfly), a6: zero point
                    accF = warp_sum(accF);
                    double S = 1.0;
                    if (g_zp != nullptr) S = exp10(0.4 * (double)g_zp[o]) * __ldg(P.band_zpab_inv + b);
                    m = S * x0 * (double)accF;
                    if (GRAD) {
                        accB = warp_sum(accB);
                        accC = warp_sum(accC);
                        accD = warp_sum(accD);
                        dm0 = S * (double)accF;
                        dm1 = S * x0 * (double)accB;
                        dm2 = S * x0 * (double)accC;
                        dm3 = -S * x0 * (double)accD * inv_opz;
                    }
                }
            }
            // ---- outputs of this evaluation
            if (lane == 0) {
                if (o_flux) o_flux[out_base + i] = (T)m;
                if (GRAD && o_dflux) {
                    V4 *dst = reinterpret_cast<V4 *>(o_dflux) + (out_base + i);
                    *dst = make_v4<T>((T)dm0, (T)dm1, (T)dm2, (T)dm3);
                }
            }
            if (want_chi) { // a7 (every lane carries the same partial)
                const double f = (double)g_flux[o], e = (double)g_err[o];
                const double rr = (f - m) / e;
                chi += rr * rr;
                if (GRAD) {
                    const double g = -2.0 * (f - m) / (e * e);
                    dchi0 += g * dm0;
                    dchi1 += g * dm1;
                    dchi2 += g * dm2;
                    dchi3 += g * dm3;
                }
            }
        }
        if (want_chi) { // fixed-order sum over warps: deterministic
            if (lane == 0) {
                red[warp * 5 + 0] = chi;
                red[warp * 5 + 1] = dchi0;
                red[warp * 5 + 2] = dchi1;
                red[warp * 5 + 3] = dchi2;
                red[warp * 5 + 4] = dchi3;
            }
            __syncthreads();
            if (tid < 5) {
                double s = 0.0;
                for (int w = 0; w < NWARPS; ++w) s += red[w * 5 + tid];
                if (tid == 0) {
                    if (P.out_chi2) static_cast<T *>(P.out_chi2)[unit] = (T)s;
                } else if (GRAD && P.out_dchi2) {
                    static_cast<T *>(P.out_dchi2)[unit * 4 + (tid - 1)] = (T)s;
                }
            }
            __syncthreads();
        }
    }
}

} // namespace sb
