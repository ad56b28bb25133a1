// sb_fit.cuh -- lane kernels of the device-resident batched L-BFGS fit driver (sb_fit_lbfgs).
//
// PAPER.md:17 names the workload ("fmin_bfgs.py ... optimisation via L-BFGS-B"); the paper gives no
// algorithmic detail, so the algorithm is the textbook one (Nocedal & Wright, Numerical Optimization:
// two-loop recursion, Alg. 7.4; backtracking line search with the Armijo condition, Alg. 3.1), in the
// reading G16 of DESIGN.md:
//   variables   u = theta / s, s = (x0 of the start point, 1, 1, 1); gradient g_u = g_theta * s.
//   one STEP of the driver = one batched evaluation of chi^2 and d chi^2/d theta at the trial point of
//   every live lane (sb_bandflux_grad's kernels) followed by sb_fit_update_kernel, which advances the
//   state machine of every lane (one thread per lane, fp64, fixed summation order):
//     first evaluation: d = -g, alpha = min(1, 1/|g|);
//     later evaluations are at u_t = P(u + alpha d) (P: projection on the box) and are ACCEPTED if
//     f_t is finite and f_t <= f + c1 g.(u_t - u), c1 = 1e-4:
//       accepted  s = u_t - u, y = g_t - g stored (circular memory) if s.y > 1e-10 |s| |y|; converged
//                 if f - f_t <= ftol max(|f|, |f_t|, 1) or max|g_t| <= gtol; d = -H g_t by the two-loop
//                 recursion with H0 = (s.y / y.y) I of the newest pair (steepest descent and an empty
//                 memory if there is no pair or g_t.d >= 0); alpha = 1;
//       rejected  alpha /= 2; 30 rejections in a row stop the lane (stalled).
//     a lane also stops after max_eval evaluations or max_iter accepted steps.
// Nothing here is shared with oracle/lbfgs.py (which restates the same algorithm in Python for the
// tests).  Products and sums are written with __dmul_rn / __dadd_rn so that the compiler cannot
// contract them into fused multiply-adds: the sequence of roundings is the one the algorithm states.
#pragma once
#include <stdint.h>

namespace sbf {

constexpr int kMaxMemory = 8;
constexpr int kMaxBacktrack = 30;
constexpr double kC1 = 1e-4;
constexpr double kCurvEps = 1e-10;

enum { ST_RUNNING = 0, ST_CONVERGED = 1, ST_STALLED = 2, ST_EXHAUSTED = 3 };

// Per-lane state in the fit workspace, structure of arrays: element k of lane i of a [4][n] array is at
// [k * n + i] (coalesced: one thread per lane).
struct FitState {
    double *u, *g, *d, *ut;      // [4][n]
    double *f, *alpha, *scale;   // [n]; scale = x0 of the start point (1 if that is 0)
    double *S, *Y;               // [memory][4][n]
    int32_t *n_hist, *head, *n_eval, *n_iter, *n_back, *status; // [n]
    int32_t *live;               // [n] 1 while the lane is running (read by the evaluation kernels)
    int32_t *n_live;             // [1] running lanes (evaluation kernels return at once when it is 0)
};

struct FitParams {
    FitState st;
    int32_t n;                   // lanes = units
    int32_t memory, max_eval, max_iter, trace_len;
    double ftol, gtol;
    double lo[4], hi[4];         // box in theta units (-inf / +inf when absent)
    int32_t has_box;
    void *x0, *x1, *c, *t0;      // [n] trial theta of the batch's element type (workspace)
    const void *chi2, *dchi2;    // [n], [n][4] results of the evaluation at the trial theta
    void *theta_out, *chi2_out;  // [n][4], [n] of the batch's element type, or NULL
    int32_t *status_out, *n_iter_out, *n_eval_out; // [n] or NULL
    double *trace_out;           // [trace_len][n] chi^2 after i accepted steps (NaN: not reached), or NULL
};

__device__ __forceinline__ double mul(double a, double b) { return __dmul_rn(a, b); }
__device__ __forceinline__ double add(double a, double b) { return __dadd_rn(a, b); }
__device__ __forceinline__ double sub(double a, double b) { return __dadd_rn(a, -b); }
__device__ __forceinline__ double dot4(const double (&a)[4], const double (&b)[4])
{
    double s = 0.0;
#pragma unroll
    for (int k = 0; k < 4; ++k) s = add(s, mul(a[k], b[k]));
    return s;
}

__device__ __forceinline__ void project(const FitParams &F, const double (&sc)[4], double (&v)[4])
{
    if (!F.has_box) return;
#pragma unroll
    for (int k = 0; k < 4; ++k) { // bounds are given in theta units; the lane works in u = theta / s
        double a = F.lo[k] / sc[k], b = F.hi[k] / sc[k];
        if (sc[k] < 0.0) { const double t = a; a = b; b = t; }
        v[k] = fmin(fmax(v[k], a), b);
    }
}

// theta_k = u_k s_k in the batch's element type, INSIDE the box: the projection above works in u, and both
// (lo/s) s and the rounding to T can land one ulp outside [lo, hi]; clamp in theta units and, where the cast
// crosses a bound, step to the neighbouring value of T on the inside.
template <typename T> __device__ __forceinline__ T to_theta(const FitParams &F, int k, double u, double s)
{
    double th = mul(u, s);
    if (!F.has_box) return (T)th;
    th = fmin(fmax(th, F.lo[k]), F.hi[k]);
    T r = (T)th;
    if constexpr (sizeof(T) == 4) {
        if ((double)r < F.lo[k]) r = nextafterf(r, INFINITY);
        else if ((double)r > F.hi[k]) r = nextafterf(r, -INFINITY);
    }
    return r;
}

template <typename T> __device__ __forceinline__ void store_theta(const FitParams &F, int i, const double (&v)[4], const double (&sc)[4])
{
    static_cast<T *>(F.x0)[i] = to_theta<T>(F, 0, v[0], sc[0]);
    static_cast<T *>(F.x1)[i] = to_theta<T>(F, 1, v[1], sc[1]);
    static_cast<T *>(F.c)[i] = to_theta<T>(F, 2, v[2], sc[2]);
    static_cast<T *>(F.t0)[i] = to_theta<T>(F, 3, v[3], sc[3]);
}

// Start: u = P(theta_start / s), trial theta = u s; every lane live.
template <typename T>
__global__ void __launch_bounds__(256) sb_fit_init_kernel(const FitParams F, const T *__restrict__ x0, const T *__restrict__ x1,
                                                          const T *__restrict__ c, const T *__restrict__ t0)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i == 0) *F.st.n_live = F.n;
    if (i >= F.n) return;
    const int n = F.n;
    const double th[4] = {(double)x0[i], (double)x1[i], (double)c[i], (double)t0[i]};
    const double s0 = th[0] != 0.0 ? th[0] : 1.0;
    const double sc[4] = {s0, 1.0, 1.0, 1.0};
    double u[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) u[k] = th[k] / sc[k];
    project(F, sc, u);
    F.st.scale[i] = s0;
#pragma unroll
    for (int k = 0; k < 4; ++k) { F.st.u[k * n + i] = u[k]; F.st.ut[k * n + i] = u[k]; }
    store_theta<T>(F, i, u, sc);
    F.st.n_hist[i] = 0; F.st.head[i] = 0; F.st.n_eval[i] = 0; F.st.n_iter[i] = 0; F.st.n_back[i] = 0;
    F.st.status[i] = ST_RUNNING;
    F.st.live[i] = 1;
    if (F.trace_out)
        for (int t = 0; t < F.trace_len; ++t) F.trace_out[(size_t)t * n + i] = __longlong_as_double(0x7ff8000000000000LL);
}

// One step of every running lane after the evaluation at its trial point.
template <typename T> __global__ void __launch_bounds__(128) sb_fit_update_kernel(const FitParams F)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= F.n) return;
    const FitState &st = F.st;
    if (st.status[i] != ST_RUNNING) return;
    const int n = F.n;
    const double s0 = st.scale[i];
    const double sc[4] = {s0, 1.0, 1.0, 1.0};
    const double ft = (double)static_cast<const T *>(F.chi2)[i];
    double gt[4], u[4], g[4], d[4], ut[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        gt[k] = mul((double)static_cast<const T *>(F.dchi2)[4 * (size_t)i + k], sc[k]);
        u[k] = st.u[k * n + i];
        ut[k] = st.ut[k * n + i];
    }
    int n_eval = st.n_eval[i], n_iter = st.n_iter[i], n_back = st.n_back[i];
    int status = ST_RUNNING;
    double f, alpha;
    auto steepest = [&]() { // d = -g, alpha = min(1, 1/|g|); empties the memory
#pragma unroll
        for (int k = 0; k < 4; ++k) d[k] = -g[k];
        const double gn = sqrt(dot4(g, g));
        alpha = gn > 0.0 ? fmin(1.0, 1.0 / gn) : 1.0;
        st.n_hist[i] = 0;
        return gn;
    };
    if (n_eval == 0) { // evaluation at the start point
        n_eval = 1;
        f = ft;
#pragma unroll
        for (int k = 0; k < 4; ++k) g[k] = gt[k];
        if (F.trace_out && F.trace_len > 0) F.trace_out[i] = f;
        if (!isfinite(f)) status = ST_STALLED;
        const double gn = steepest();
        const double gmax = fmax(fmax(fabs(g[0]), fabs(g[1])), fmax(fabs(g[2]), fabs(g[3])));
        if (status == ST_RUNNING && (gn == 0.0 || gmax <= F.gtol)) status = ST_CONVERGED;
    } else {
        n_eval += 1;
        f = st.f[i];
        alpha = st.alpha[i];
        double step[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            g[k] = st.g[k * n + i];
            d[k] = st.d[k * n + i];
            step[k] = sub(ut[k], u[k]);
        }
        if (isfinite(ft) && ft <= add(f, mul(kC1, dot4(g, step)))) { // Armijo: accepted
            double y[4];
#pragma unroll
            for (int k = 0; k < 4; ++k) y[k] = sub(gt[k], g[k]);
            const double sy = dot4(step, y);
            int cnt = st.n_hist[i], head = st.head[i];
            if (sy > mul(mul(kCurvEps, sqrt(dot4(step, step))), sqrt(dot4(y, y)))) { // curvature pair kept
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    st.S[((size_t)head * 4 + k) * n + i] = step[k];
                    st.Y[((size_t)head * 4 + k) * n + i] = y[k];
                }
                head = head + 1 == F.memory ? 0 : head + 1;
                if (cnt < F.memory) ++cnt;
                st.head[i] = head;
                st.n_hist[i] = cnt;
            }
            const double gmax = fmax(fmax(fabs(gt[0]), fabs(gt[1])), fmax(fabs(gt[2]), fabs(gt[3])));
            const bool done = sub(f, ft) <= mul(F.ftol, fmax(fmax(fabs(f), fabs(ft)), 1.0)) || gmax <= F.gtol;
            f = ft;
#pragma unroll
            for (int k = 0; k < 4; ++k) { u[k] = ut[k]; g[k] = gt[k]; }
            n_iter += 1;
            n_back = 0;
            if (F.trace_out && n_iter < F.trace_len) F.trace_out[(size_t)n_iter * n + i] = f;
            if (done) {
                status = ST_CONVERGED;
            } else {
                bool reset = cnt == 0;
                if (!reset) { // two-loop recursion over the stored pairs, newest first then oldest first
                    double q[4], al[kMaxMemory], rho[kMaxMemory];
#pragma unroll
                    for (int k = 0; k < 4; ++k) q[k] = g[k];
                    auto pair = [&](int j, double (&s)[4], double (&yy)[4]) { // j-th oldest pair
                        int slot = head - cnt + j;
                        if (slot < 0) slot += F.memory;
#pragma unroll
                        for (int k = 0; k < 4; ++k) {
                            s[k] = st.S[((size_t)slot * 4 + k) * n + i];
                            yy[k] = st.Y[((size_t)slot * 4 + k) * n + i];
                        }
                    };
                    double s[4], yy[4];
                    for (int j = cnt - 1; j >= 0; --j) {
                        pair(j, s, yy);
                        rho[j] = 1.0 / dot4(yy, s);
                        al[j] = mul(rho[j], dot4(s, q));
#pragma unroll
                        for (int k = 0; k < 4; ++k) q[k] = sub(q[k], mul(al[j], yy[k]));
                    }
                    pair(cnt - 1, s, yy);
                    const double gamma = dot4(s, yy) / dot4(yy, yy);
                    double r[4];
#pragma unroll
                    for (int k = 0; k < 4; ++k) r[k] = mul(gamma, q[k]);
                    for (int j = 0; j < cnt; ++j) {
                        pair(j, s, yy);
                        const double beta = mul(rho[j], dot4(yy, r));
                        const double co = sub(al[j], beta);
#pragma unroll
                        for (int k = 0; k < 4; ++k) r[k] = add(r[k], mul(co, s[k]));
                    }
#pragma unroll
                    for (int k = 0; k < 4; ++k) d[k] = -r[k];
                    if (dot4(g, d) >= 0.0) reset = true;
                }
                if (reset) steepest();
                else alpha = 1.0;
            }
        } else { // rejected: halve the step
            alpha = mul(alpha, 0.5);
            n_back += 1;
            if (n_back >= kMaxBacktrack) status = ST_STALLED;
        }
    }
    if (status == ST_RUNNING && (n_eval >= F.max_eval || n_iter >= F.max_iter)) status = ST_EXHAUSTED;
    if (status == ST_RUNNING) { // next trial point
#pragma unroll
        for (int k = 0; k < 4; ++k) ut[k] = add(u[k], mul(alpha, d[k]));
        project(F, sc, ut);
        store_theta<T>(F, i, ut, sc);
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            st.u[k * n + i] = u[k];
            st.g[k * n + i] = g[k];
            st.d[k * n + i] = d[k];
            st.ut[k * n + i] = ut[k];
        }
        st.f[i] = f;
        st.alpha[i] = alpha;
    } else { // the lane stops: its result is the last accepted point
        st.live[i] = 0;
        atomicSub(st.n_live, 1);
        if (F.theta_out) {
            T *o = static_cast<T *>(F.theta_out) + 4 * (size_t)i;
#pragma unroll
            for (int k = 0; k < 4; ++k) o[k] = to_theta<T>(F, k, u[k], sc[k]);
        }
        if (F.chi2_out) static_cast<T *>(F.chi2_out)[i] = (T)f;
        if (F.status_out) F.status_out[i] = status;
        if (F.n_iter_out) F.n_iter_out[i] = n_iter;
        if (F.n_eval_out) F.n_eval_out[i] = n_eval;
    }
    st.n_eval[i] = n_eval;
    st.n_iter[i] = n_iter;
    st.n_back[i] = n_back;
    st.status[i] = status;
}

} // namespace sbf
