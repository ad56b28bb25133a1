// saltband.cu -- C ABI of libsaltband (include/saltband.h): loaders, argument checks, launches.
// Product code; shares nothing with oracle/.  Build: see paper_2504_08081_b200/build.py.
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>
#include <type_traits>
#include <vector>

#include <nvtx3/nvToolsExt.h>

#include "sb_internal.h"
#include "sb_kernels.cuh"
#include "sb_hoist.cuh"
#include "sb_nw.cuh"
#include "sb_fit.cuh"

// Per-stream workspaces and host-call contexts of a bands handle.  This is the only mutable state
// behind the handles: a cache, guarded by `mu`.  A compute call without a pack needs a few hundred KB
// of scratch (z-order permutation, sort counters); it is taken from the slot of the call's stream,
// which the handle allocates on the first call on that stream (or when a larger batch arrives) and
// keeps until sb_free_bands.  Calls on distinct streams never share a slot; calls on the same stream
// are ordered by the stream.  Replaced buffers are retired, not freed: earlier work may still use them.
struct SbScratch {
    struct Slot { cudaStream_t stream; int kind; unsigned char *buf; size_t bytes; };
    struct HostCtx { // one per concurrent host-buffer call: three streams and their staging slabs
        cudaStream_t st[3];
        unsigned char *slab[3];
        size_t slab_bytes;
        unsigned char *fit_slab; // sb_fit_lbfgs_host: the whole batch, resident for the duration of the fit
        size_t fit_bytes;
        bool busy;
    };
    std::mutex mu;
    std::vector<Slot> slots;
    std::vector<void *> retired;
    std::vector<HostCtx *> host;
};

struct NvtxRange { // NVTX range around every sb_* call
    explicit NvtxRange(const char *name) { nvtxRangePushA(name); }
    ~NvtxRange() { nvtxRangePop(); }
};

namespace {

thread_local int32_t tl_launches = 0;
thread_local int32_t tl_cuda_err = 0;
thread_local int32_t tl_form = 0;

bool cuda_ok(cudaError_t e)
{
    if (e == cudaSuccess) return true;
    tl_cuda_err = (int32_t)e;
    return false;
}

template <typename T> bool upload(T **dst, const std::vector<T> &src)
{
    *dst = nullptr;
    size_t bytes = src.size() * sizeof(T);
    if (bytes == 0) bytes = sizeof(T);
    if (!cuda_ok(cudaMalloc((void **)dst, bytes))) return false;
    if (!src.empty() && !cuda_ok(cudaMemcpy(*dst, src.data(), src.size() * sizeof(T), cudaMemcpyHostToDevice)))
        return false;
    return true;
}

bool uniform_increasing(const double *x, int32_t n)
{
    if (n < 2) return false;
    for (int32_t i = 0; i < n; ++i)
        if (!std::isfinite(x[i])) return false;
    const double step = (x[n - 1] - x[0]) / (double)(n - 1);
    if (!(step > 0.0)) return false;
    for (int32_t i = 1; i < n; ++i) {
        const double d = x[i] - x[i - 1];
        if (!(d > 0.0) || std::fabs(d - step) > 1e-9 * step) return false;
    }
    return true;
}

double poly_val(const double *a, int n, double x)
{
    double s = 0.0;
    for (int q = n - 1; q >= 0; --q) s = s * x + a[q];
    return s;
}
double poly_der(const double *a, int n, double x)
{
    double s = 0.0;
    for (int q = n - 1; q >= 1; --q) s = s * x + (double)q * a[q];
    return s;
}

bool device_limits(int *n_sm, int *smem_optin)
{
    int dev = 0;
    if (!cuda_ok(cudaGetDevice(&dev))) return false;
    if (!cuda_ok(cudaDeviceGetAttribute(n_sm, cudaDevAttrMultiProcessorCount, dev))) return false;
    if (!cuda_ok(cudaDeviceGetAttribute(smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev))) return false;
    return true;
}

// Opt-in dynamic shared memory of a kernel: set once per (kernel, device) to the device maximum.
// `carve`: also prefer the largest shared-memory carveout (kernels that fill shared memory; the others keep
// the default split so that their model-table reads stay in L1).
bool allow_max_smem(const void *kern, int device, int smem_optin, bool carve = false)
{
    static std::mutex mu;
    static std::vector<std::pair<const void *, int>> done;
    std::lock_guard<std::mutex> lock(mu);
    for (const auto &d : done)
        if (d.first == kern && d.second == device) return true;
    cudaFuncAttributes fa;
    if (!cuda_ok(cudaFuncGetAttributes(&fa, kern))) return false;
    const int dyn = smem_optin - (int)fa.sharedSizeBytes; // static + dynamic <= the opt-in limit
    if (!cuda_ok(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, dyn))) return false;
    if (carve) cudaFuncSetAttribute(kern, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
    done.emplace_back(kern, device);
    return true;
}

// Workspace of at least `bytes` for calls on `stream` (see SbScratch).  Allocates only when the stream
// has no slot yet or its slot is too small.
enum { kScratchSort = 0, kScratchFit = 1 }; // what a slot is for: calls of different kinds may nest
unsigned char *scratch_for(const sb_bands *b, cudaStream_t stream, size_t bytes, int kind = kScratchSort)
{
    SbScratch *sc = b->scratch;
    std::lock_guard<std::mutex> lock(sc->mu);
    for (auto &s : sc->slots)
        if (s.stream == stream && s.kind == kind) {
            if (s.bytes >= bytes) return s.buf;
            unsigned char *nb = nullptr;
            const size_t want = bytes + bytes / 2;
            if (!cuda_ok(cudaMalloc((void **)&nb, want))) return nullptr;
            sc->retired.push_back(s.buf);
            s.buf = nb;
            s.bytes = want;
            return nb;
        }
    unsigned char *nb = nullptr;
    if (!cuda_ok(cudaMalloc((void **)&nb, bytes))) return nullptr;
    sc->slots.push_back({stream, kind, nb, bytes});
    return nb;
}

} // namespace

extern "C" {

const char *sb_version(void) { return "saltband 0.2 (sm_100a)"; }

const char *sb_strerror(int status)
{
    switch (status) {
    case SB_OK: return "ok";
    case SB_EINVAL: return "invalid argument";
    case SB_ENOMEM: return "out of memory";
    case SB_ECUDA: return "CUDA error (no device, or a copy/launch failed)";
    case SB_ELIMIT: return "table exceeds on-chip staging limits";
    default: return "unknown status";
    }
}

int32_t sb_last_launch_count(void) { return tl_launches; }
int32_t sb_last_cuda_error(void) { return tl_cuda_err; }
int32_t sb_last_form(void) { return tl_form; }

int sb_load_model(const double *phase, int32_t n_phase, const double *wave, int32_t n_wave, const double *m0,
                  const double *m1, const double *cl_coef, int32_t n_cl, double cl_wave_b, double cl_wave_v,
                  double cl_lo, double cl_hi, sb_model **out)
{
    NvtxRange nvtx("sb_load_model");
    if (out) *out = nullptr;
    if (!phase || !wave || !m0 || !m1 || !cl_coef || !out) return SB_EINVAL;
    if (n_phase < 2 || n_wave < 2 || n_cl < 1 || n_cl > SB_MAX_CL) return SB_EINVAL;
    if (!uniform_increasing(phase, n_phase) || !uniform_increasing(wave, n_wave)) return SB_EINVAL;
    if (!std::isfinite(cl_wave_b) || !std::isfinite(cl_wave_v) || cl_wave_b == cl_wave_v) return SB_EINVAL;
    if (!std::isfinite(cl_lo) || !std::isfinite(cl_hi) || !(cl_lo < cl_hi)) return SB_EINVAL;
    for (int q = 0; q < n_cl; ++q)
        if (!std::isfinite(cl_coef[q])) return SB_EINVAL;
    const size_t n = (size_t)n_phase * (size_t)n_wave;
    for (size_t i = 0; i < n; ++i)
        if (!std::isfinite(m0[i]) || !std::isfinite(m1[i])) return SB_EINVAL;
    if ((long long)n_phase * ((long long)n_wave + SB_PAD_L + SB_PAD_R + 4) >= (1LL << 30)) return SB_ELIMIT;

    sb_model *h = new (std::nothrow) sb_model();
    if (!h) return SB_ENOMEM;
    memset(h, 0, sizeof(*h));
    SbModelParams &p = h->prm;
    p.n_phase = n_phase;
    p.n_wave = n_wave;
    p.ld = (n_wave + SB_PAD_L + SB_PAD_R + 3) & ~3; // zero columns left and right of the nodes (sb_internal.h)
    p.n_cl = n_cl;
    p.p0 = phase[0];
    p.dp = (phase[n_phase - 1] - phase[0]) / (double)(n_phase - 1);
    p.inv_dp = 1.0 / p.dp;
    p.l0 = wave[0];
    p.dl = (wave[n_wave - 1] - wave[0]) / (double)(n_wave - 1);
    for (int q = 0; q < SB_MAX_CL; ++q) p.cl[q] = q < n_cl ? cl_coef[q] : 0.0;
    p.cl_b = cl_wave_b;
    p.cl_inv_span = 1.0 / (cl_wave_v - cl_wave_b);
    double r_lo = (cl_lo - cl_wave_b) * p.cl_inv_span, r_hi = (cl_hi - cl_wave_b) * p.cl_inv_span;
    if (r_lo > r_hi) { double t = r_lo; r_lo = r_hi; r_hi = t; } // cl_wave_v < cl_wave_b flips the axis
    p.r_lo = r_lo;
    p.r_hi = r_hi;
    p.p_lo = poly_val(p.cl, n_cl, r_lo);
    p.s_lo = poly_der(p.cl, n_cl, r_lo);
    p.p_hi = poly_val(p.cl, n_cl, r_hi);
    p.s_hi = poly_der(p.cl, n_cl, r_hi);

    std::vector<double> t0((size_t)n_phase * p.ld, 0.0), t1((size_t)n_phase * p.ld, 0.0);
    for (int k = 0; k < n_phase; ++k)
        for (int l = 0; l < n_wave; ++l) {
            t0[(size_t)k * p.ld + SB_PAD_L + l] = m0[(size_t)k * n_wave + l];
            t1[(size_t)k * p.ld + SB_PAD_L + l] = m1[(size_t)k * n_wave + l];
        }
    std::vector<float> f0(t0.begin(), t0.end()), f1(t1.begin(), t1.end());
    cudaGetDevice(&h->device);
    if (!device_limits(&h->n_sm, &h->smem_optin)) { delete h; return SB_ECUDA; }
    if (!upload(&h->m0_f64, t0) || !upload(&h->m1_f64, t1) || !upload(&h->m0_f32, f0) || !upload(&h->m1_f32, f1)) {
        sb_free_model(h);
        return tl_cuda_err == (int32_t)cudaErrorMemoryAllocation ? SB_ENOMEM : SB_ECUDA;
    }
    if (n_wave + 48 <= SBH_LDN && n_phase >= 4) { // interleaved {M0, M1} table of the band-grouped kernel
        std::vector<float2> t01((size_t)n_phase * SBH_LDN, make_float2(0.f, 0.f));
        for (int k = 0; k < n_phase; ++k)
            for (int l = 0; l < n_wave; ++l)
                t01[(size_t)k * SBH_LDN + SBH_PAD_L + l] =
                    make_float2((float)m0[(size_t)k * n_wave + l], (float)m1[(size_t)k * n_wave + l]);
        if (!upload(&h->m01_f32, t01)) {
            sb_free_model(h);
            return tl_cuda_err == (int32_t)cudaErrorMemoryAllocation ? SB_ENOMEM : SB_ECUDA;
        }
    }
    if ((size_t)n_phase * p.ld * sizeof(float) <= (size_t)SBN_M1_OFF) { // tables of the node-weight kernel (sb_internal.h)
        const size_t m1_at = SBN_M1_OFF / sizeof(float);
        std::vector<float> tx(m1_at + (size_t)n_phase * p.ld, 0.f);
        for (int k = 0; k < n_phase; ++k)
            for (int l = 0; l < n_wave; ++l) {
                const size_t at = (size_t)k * p.ld + SB_PAD_L + l;
                tx[at] = (float)m0[(size_t)k * n_wave + l];
                tx[m1_at + at] = (float)m1[(size_t)k * n_wave + l];
            }
        if (!upload(&h->mx_f32, tx)) {
            sb_free_model(h);
            return tl_cuda_err == (int32_t)cudaErrorMemoryAllocation ? SB_ENOMEM : SB_ECUDA;
        }
    }
    // the uploads above are cudaMemcpy from pageable memory (they may return once the data is staged): make the
    // tables complete before a compute call on a non-blocking stream, which is not ordered after them, reads them
    if (!cuda_ok(cudaDeviceSynchronize())) { sb_free_model(h); return SB_ECUDA; }
    *out = h;
    return SB_OK;
}

void sb_free_model(sb_model *m)
{
    if (!m) return;
    cudaFree(m->m0_f32);
    cudaFree(m->m1_f32);
    cudaFree(m->m0_f64);
    cudaFree(m->m1_f64);
    cudaFree(m->m01_f32);
    cudaFree(m->mx_f32);
    delete m;
}

int sb_load_bandpasses(int32_t n_bands, const int64_t *offset, const double *wave, const double *trans,
                       sb_bands **out)
{
    NvtxRange nvtx("sb_load_bandpasses");
    if (out) *out = nullptr;
    if (!offset || !wave || !trans || !out || n_bands < 1) return SB_EINVAL;
    if (offset[0] != 0) return SB_EINVAL;
    for (int b = 0; b < n_bands; ++b)
        if (offset[b + 1] - offset[b] < 2) return SB_EINVAL;
    const int64_t total = offset[n_bands];
    if (total >= (1LL << 30)) return SB_ELIMIT;
    for (int64_t i = 0; i < total; ++i)
        if (!std::isfinite(wave[i]) || !std::isfinite(trans[i]) || !(wave[i] > 0.0)) return SB_EINVAL;
    for (int b = 0; b < n_bands; ++b)
        for (int64_t i = offset[b] + 1; i < offset[b + 1]; ++i)
            if (!(wave[i] > wave[i - 1])) return SB_EINVAL;

    sb_bands *h = new (std::nothrow) sb_bands();
    if (!h) return SB_ENOMEM;
    memset(h, 0, sizeof(*h));
    h->n_bands = n_bands;
    h->n_total = (int32_t)total;
    h->h_zpab = (double *)malloc(sizeof(double) * (size_t)n_bands);
    h->scratch = new (std::nothrow) SbScratch();
    if (!h->h_zpab || !h->scratch) { free(h->h_zpab); delete h->scratch; delete h; return SB_ENOMEM; }

    const double hc = SB_H_PLANCK * SB_C_ANGSTROM;
    std::vector<int32_t> off(n_bands + 1);
    std::vector<double> lam_first(n_bands), zpab_inv(n_bands), dlam(total), w(total);
    for (int b = 0; b <= n_bands; ++b) off[b] = (int32_t)offset[b];
    for (int b = 0; b < n_bands; ++b) {
        const int64_t lo = offset[b], n = offset[b + 1] - lo;
        const double *lam = wave + lo, *tr = trans + lo;
        if ((int32_t)n > h->max_n) h->max_n = (int32_t)n;
        if (lam[n - 1] - lam[0] > h->max_span) h->max_span = lam[n - 1] - lam[0];
        lam_first[b] = lam[0];
        double zp = 0.0;
        for (int64_t j = 0; j < n; ++j) {
            // trapezoid weight of node j: half the distance between its neighbours
            const double left = j > 0 ? lam[j] - lam[j - 1] : 0.0;
            const double right = j + 1 < n ? lam[j + 1] - lam[j] : 0.0;
            const double wq = 0.5 * (left + right);
            dlam[lo + j] = lam[j] - lam[0];
            w[lo + j] = wq * tr[j] * lam[j] / hc; // folded: w_j T_j lam_j/(hc)
            zp += wq * (SB_AB_FNU * SB_C_ANGSTROM / (lam[j] * lam[j])) * tr[j] * lam[j] / hc; // G7
        }
        h->h_zpab[b] = zp;
        zpab_inv[b] = 1.0 / zp;
    }
    // uniform band grids (all of them) enable the band-grouped kernel: lam_j = lam_first + j h_b
    std::vector<double> hstep(n_bands);
    std::vector<float> w_f(w.begin(), w.end());
    h->all_uniform = 1;
    for (int b = 0; b < n_bands; ++b) {
        const int64_t lo = offset[b], n = offset[b + 1] - lo;
        const double *lam = wave + lo;
        hstep[b] = (lam[n - 1] - lam[0]) / (double)(n - 1);
        for (int64_t j = 0; j < n; ++j)
            if (std::fabs(lam[j] - (lam[0] + (double)j * hstep[b])) > 1e-9 * lam[j]) h->all_uniform = 0;
    }
    std::vector<float2> tab_f((size_t)total), wd_f((size_t)total);
    std::vector<double2> tab_d((size_t)total);
    for (int64_t i = 0; i < total; ++i) {
        tab_d[i] = make_double2(dlam[i], w[i]);
        tab_f[i] = make_float2((float)dlam[i], (float)w[i]);
    }
    for (int b = 0; b < n_bands; ++b) // offset of every sample from the band's mean-step grid (0 on uniform grids)
        for (int64_t i = offset[b]; i < offset[b + 1]; ++i)
            wd_f[i] = make_float2((float)w[i], (float)(dlam[i] - (double)(i - offset[b]) * hstep[b]));
    cudaGetDevice(&h->device);
    if (!upload(&h->d_off, off) || !upload(&h->d_lam_first, lam_first) || !upload(&h->d_zpab_inv, zpab_inv) ||
        !upload(&h->d_tab_f64, tab_d) || !upload(&h->d_tab_f32, tab_f) || !upload(&h->d_w_f32, w_f) ||
        !upload(&h->d_dlam_f64, dlam) || !upload(&h->d_h, hstep) || !upload(&h->d_wd_f32, wd_f)) {
        sb_free_bands(h);
        return tl_cuda_err == (int32_t)cudaErrorMemoryAllocation ? SB_ENOMEM : SB_ECUDA;
    }
    if (!cuda_ok(cudaDeviceSynchronize())) { sb_free_bands(h); return SB_ECUDA; } // as in sb_load_model
    *out = h;
    return SB_OK;
}

void sb_free_bands(sb_bands *b)
{
    if (!b) return;
    cudaFree(b->d_off);
    cudaFree(b->d_lam_first);
    cudaFree(b->d_zpab_inv);
    cudaFree(b->d_tab_f32);
    cudaFree(b->d_tab_f64);
    cudaFree(b->d_w_f32);
    cudaFree(b->d_wd_f32);
    cudaFree(b->d_dlam_f64);
    cudaFree(b->d_h);
    free(b->h_zpab);
    if (b->scratch) {
        for (auto &sl : b->scratch->slots) cudaFree(sl.buf);
        for (void *p : b->scratch->retired) cudaFree(p);
        for (auto *c : b->scratch->host) {
            for (int i = 0; i < 3; ++i) {
                if (c->slab[i]) cudaFree(c->slab[i]);
                if (c->st[i]) cudaStreamDestroy(c->st[i]);
            }
            if (c->fit_slab) cudaFree(c->fit_slab);
            delete c;
        }
        delete b->scratch;
    }
    delete b;
}

int32_t sb_bands_count(const sb_bands *b) { return b ? b->n_bands : 0; }
double sb_bands_zpab(const sb_bands *b, int32_t band)
{
    if (!b || band < 0 || band >= b->n_bands) return NAN;
    return b->h_zpab[band];
}

} // extern "C"

// ------------------------------------------------------------------------------------------
// Launch
// ------------------------------------------------------------------------------------------
namespace {

template <typename T, bool GRAD, int NCL, bool STAGE, int NWARPS>
int launch_inst(const sb_model *m, const SbKParams &kp, size_t smem, int grid, cudaStream_t st)
{
    auto kern = sb::sb_fused_kernel<T, GRAD, NCL, STAGE, NWARPS>;
    if (!allow_max_smem((const void *)kern, m->device, m->smem_optin)) return SB_ECUDA;
    kern<<<grid, NWARPS * 32, smem, st>>>(kp);
    if (!cuda_ok(cudaGetLastError())) return SB_ECUDA;
    tl_launches += 1;
    tl_form = SB_FORM_DIRECT;
    return SB_OK;
}

template <typename T, bool GRAD, int NWARPS>
int launch_typed(const sb_model *m, SbKParams &kp, const sb_bands *b, int n_obs_total, cudaStream_t st)
{
    const int smem_max = m->smem_optin, n_sm = m->n_sm;
    constexpr int NSET = GRAD ? 3 : 1;
    const size_t cell_bytes = sizeof(T) * 4 * NSET;
    // evaluation records per chunk and units per group: about `cap` evaluations per CTA pass
    const int cap = GRAD ? 256 : 512;
    const double mean_obs = kp.n_sn > 0 ? (double)n_obs_total / (double)kp.n_sn : 1.0;
    int group = (int)((double)cap / (mean_obs > 1.0 ? mean_obs : 1.0));
    if (group < 1) group = 1;
    if (group > sb::kMaxGroup) group = sb::kMaxGroup;
    kp.chunk_cap = cap;
    kp.group_units = group;
    // entries needed by the widest band at z >= 0 (narrower tiles still work: the kernel loops)
    int tc_full = (int)std::ceil(b->max_span / kp.mp.dl) + 12;
    if (tc_full > kp.mp.n_wave + 12) tc_full = kp.mp.n_wave + 12;
    tc_full = (tc_full + 7) & ~7;
    if (tc_full < 64) tc_full = 64;
    if (tc_full > 360) tc_full = 360; // kPassesPerTile collapse passes of 120 entries per tile
    // stage the band tables in shared memory when they fit beside >= 128-entry row buffers (fp32 only)
    const sb::SmemLayout<T, GRAD> fixed(NWARPS, 0, cap, b->n_total, false);
    const size_t band_bytes = sb::SmemLayout<T, GRAD>(NWARPS, 0, cap, b->n_total, true).total - fixed.total;
    const bool stage = sizeof(T) == 4 && fixed.total + band_bytes + (size_t)NWARPS * 128 * cell_bytes <= (size_t)smem_max;
    const size_t avail = (size_t)smem_max - fixed.total - (stage ? band_bytes : 0);
    int tc = (int)(avail / ((size_t)NWARPS * cell_bytes));
    tc &= ~7;
    if (tc > tc_full) tc = tc_full;
    if (tc < 64) return SB_ELIMIT;
    kp.tile_cells = tc;
    const size_t smem = sb::SmemLayout<T, GRAD>(NWARPS, tc, cap, b->n_total, stage).total;
    const long long n_units = (long long)kp.n_sn * kp.n_samples;
    const long long n_groups = (n_units + group - 1) / group;
    int grid = (int)(n_groups < (long long)n_sm ? n_groups : (long long)n_sm);
    if (grid < 1) return SB_OK;
    const bool small_cl = kp.mp.n_cl <= 5;
    if (stage) {
        if (small_cl) return launch_inst<T, GRAD, 5, sizeof(T) == 4, NWARPS>(m, kp, smem, grid, st);
        return launch_inst<T, GRAD, SB_MAX_CL, sizeof(T) == 4, NWARPS>(m, kp, smem, grid, st);
    }
    if (small_cl) return launch_inst<T, GRAD, 5, false, NWARPS>(m, kp, smem, grid, st);
    return launch_inst<T, GRAD, SB_MAX_CL, false, NWARPS>(m, kp, smem, grid, st);
}

// Workspace layout of the z-order sort: [0] group counter (grouped kernel), [256] bin totals, [4096]
// permutation, then the per-segment bin counts.
struct ZWork {
    size_t perm_off, hist_off, bytes;
    explicit ZWork(int n_sn)
    {
        perm_off = 4096;
        hist_off = perm_off + ((sizeof(int32_t) * (size_t)n_sn + 255) & ~(size_t)255);
        bytes = hist_off + sizeof(uint32_t) * (size_t)sbh::kZSegs * sbh::kZBins;
    }
};
static_assert(256 + sizeof(uint32_t) * sbh::kZBins <= 4096, "bin totals overlap the permutation");

// Stable z-order permutation of the supernovae into ws (one or two small kernels + a 4 KB memset).
int enqueue_zorder(const float *z, int n_sn, unsigned char *ws, cudaStream_t st, int32_t *launches)
{
    const ZWork zw(n_sn);
    unsigned int *counter = reinterpret_cast<unsigned int *>(ws);
    int32_t *perm = reinterpret_cast<int32_t *>(ws + zw.perm_off);
    if (n_sn <= sbh::kZSmall) {
        sbh::sb_zorder_small_kernel<<<1, 512, 0, st>>>(z, n_sn, perm, counter);
        if (!cuda_ok(cudaGetLastError())) return SB_ECUDA;
        *launches += 1;
        return SB_OK;
    }
    uint32_t *z_tot = reinterpret_cast<uint32_t *>(ws + 256), *z_hist = reinterpret_cast<uint32_t *>(ws + zw.hist_off);
    if (!cuda_ok(cudaMemsetAsync(ws, 0, zw.perm_off, st))) return SB_ECUDA;
    sbh::sb_zhist_kernel<<<sbh::kZCtas, sbh::kZWarps * 32, 0, st>>>(z, n_sn, z_hist, z_tot, counter);
    sbh::sb_zscatter_kernel<<<sbh::kZCtas, sbh::kZWarps * 32, 0, st>>>(z, n_sn, z_hist, z_tot, perm);
    if (!cuda_ok(cudaGetLastError())) return SB_ECUDA;
    *launches += 2;
    return SB_OK;
}

// Band-grouped kernel (sb_hoist.cuh): fp32 forward, uniform band grids.  Returns 1 when it does not
// apply (the caller then tries the next formulation), SB_OK or an error otherwise.
int launch_hoist(const sb_model *m, const sb_bands *b, const sb_batch *bt, const void *flux, const void *fluxerr,
                 void *out_flux, void *out_chi2, cudaStream_t st)
{
    constexpr int NCL = 5;
    if (!b->all_uniform || m->prm.n_cl > NCL || b->n_bands > 64 || !m->m01_f32) return 1;
    const int smem_max = m->smem_optin, n_sm = m->n_sm;
    const long long n_units = (long long)bt->n_sn * bt->n_samples;
    const double mean_obs = bt->n_sn > 0 ? (double)bt->n_obs_total / (double)bt->n_sn : 1.0;
    const int gmax = sbh::kMaxSeg, cap = 4096;
    const size_t smem = sbh::HSmem(b->n_total, cap).total;
    if (smem > (size_t)smem_max || smem > 100 * 1024) return 1;
    long long g = 1;
    double best = 0.0;
    for (long long c = 1; c <= gmax; ++c) { // busiest CTA: ceil(n_groups / n_sm) groups of about g + 4 unit-times
        if (c > 1 && (double)c * mean_obs > (double)cap) break;
        const long long ng = (n_units + c - 1) / c;
        const double load = (double)((ng + n_sm - 1) / n_sm) * (double)(c + 4);
        if (c == 1 || load <= best) { best = load; g = c; }
    }
    const ZWork zw(bt->n_sn);
    unsigned char *ws = scratch_for(b, st, zw.bytes);
    if (!ws) return tl_cuda_err == (int32_t)cudaErrorMemoryAllocation ? SB_ENOMEM : SB_ECUDA;
    SbHParams hp;
    memset(&hp, 0, sizeof(hp));
    hp.mp = m->prm;
    hp.m01 = m->m01_f32;
    hp.m0 = m->m0_f32;
    hp.m1 = m->m1_f32;
    hp.n_bands = b->n_bands;
    hp.n_band_total = b->n_total;
    hp.band_off = b->d_off;
    hp.band_lam_first = b->d_lam_first;
    hp.band_zpab_inv = b->d_zpab_inv;
    hp.band_h = b->d_h;
    hp.band_dlam = b->d_dlam_f64;
    hp.band_w = b->d_w_f32;
    hp.n_sn = bt->n_sn;
    hp.n_samples = bt->n_samples;
    hp.obs_offset = bt->obs_offset;
    hp.time = (const float *)bt->time;
    hp.zp = (const float *)bt->zp;
    hp.z = (const float *)bt->z;
    hp.x0 = (const float *)bt->x0;
    hp.x1 = (const float *)bt->x1;
    hp.c = (const float *)bt->c;
    hp.t0 = (const float *)bt->t0;
    hp.band = bt->band;
    hp.flux = (const float *)flux;
    hp.fluxerr = (const float *)fluxerr;
    hp.out_flux = (float *)out_flux;
    hp.out_chi2 = (float *)out_chi2;
    hp.counter = reinterpret_cast<unsigned int *>(ws);
    hp.perm = reinterpret_cast<const int32_t *>(ws + zw.perm_off);
    hp.group_units = (int)g;
    hp.cap = cap;
    int rc = enqueue_zorder(hp.z, hp.n_sn, ws, st, &tl_launches);
    if (rc != SB_OK) return rc;
    const long long n_groups = (n_units + g - 1) / g;
    const int grid = (int)(n_groups < (long long)n_sm ? n_groups : (long long)n_sm);
    auto kern = sbh::sb_hoist_kernel<NCL, SBH_LDN>;
    if (!allow_max_smem((const void *)kern, m->device, m->smem_optin)) return SB_ECUDA;
    kern<<<grid, sbh::kThreads, smem, st>>>(hp);
    if (!cuda_ok(cudaGetLastError())) return SB_ECUDA;
    tl_launches += 1;
    tl_form = SB_FORM_GROUPED;
    return SB_OK;
}

// Fit driver only: per-unit "live" flags and their count, written by the lane kernels (sb_fit.cuh) and
// read by the evaluation kernels, which skip the units of stopped lanes and return at once when no lane
// is left.
struct RunLive { const int32_t *live = nullptr, *n_live = nullptr; };

template <int NCL, bool GRAD, bool NU>
int launch_nw_inst(const sb_model *m, const sbn::SbNParams &np, size_t smem, int grid, cudaStream_t st)
{
    auto kern = sbn::sb_nw_kernel<NCL, GRAD, NU>;
    if (!allow_max_smem((const void *)kern, m->device, m->smem_optin, true)) return SB_ECUDA;
    kern<<<grid, 16 * 32, smem, st>>>(np);
    if (!cuda_ok(cudaGetLastError())) return SB_ECUDA;
    tl_launches += 1;
    tl_form = SB_FORM_TILED;
    return SB_OK;
}

// Node-weight kernel (sb_nw.cuh): fp32 forward and gradient, uniform band grids.  With a pack nothing is
// computed here but the launch geometry; without one the z-order permutation is built in the call's
// stream workspace first and the item geometry is computed inside the kernel.  Returns 1 when the
// kernel does not apply.
int launch_nw(bool grad, const sb_model *m, const sb_bands *b, const sb_batch *bt, const void *flux,
              const void *fluxerr, void *out_flux, void *out_chi2, void *out_dflux, void *out_dchi2, cudaStream_t st,
              const RunLive &lv)
{
    if (m->prm.n_cl > SB_MAX_CL || b->n_bands > sbn::kMaxBands || !m->mx_f32) return 1;
    if (m->prm.n_phase < 4 || m->prm.n_phase > 4096) return 1;
    const int smem_max = m->smem_optin, n_sm = m->n_sm;
    const long long n_units = (long long)bt->n_sn * bt->n_samples;
    const double mean_obs = bt->n_sn > 0 ? (double)bt->n_obs_total / (double)bt->n_sn : 1.0;
    const bool nu = !b->all_uniform; // non-uniform band grids: the kernel variant that reads {W_j, delta_j}
    // one CTA of 16 warps per SM; observations per round: as many as fit beside the band tables
    constexpr int nw = 16;
    const int nsl = grad ? nw : 2 * nw;
    int cap = grad ? sbn::Cfg<16>::kCapGrad : sbn::Cfg<16>::kCapFwd;
    while (cap >= 512 && sbn::NSmem(b->n_total, cap, grad, b->n_bands * nsl, nw, nu).total > (size_t)smem_max) cap -= 128;
    if (cap < 512) return 1;
    const size_t smem = sbn::NSmem(b->n_total, cap, grad, b->n_bands * nsl, nw, nu).total;
    const int n_cta = n_sm; // resident CTAs
    // groups: whole waves of n_sm groups of at most g_target units (even split of the z-ordered units),
    // g_target = as many units as fit the item slots and the round's observation capacity
    long long g_target = (long long)((double)cap / (mean_obs > 1.0 ? mean_obs : 1.0));
    if (g_target > nsl) g_target = nsl;
    if (g_target < 1) g_target = 1;
    long long waves = (n_units + g_target * n_cta - 1) / (g_target * n_cta);
    long long n_groups = waves * n_cta;
    if (n_groups > n_units) n_groups = n_units;
    if (n_groups < 1) return SB_OK;

    const sb_pack *pk = bt->pack;
    const int32_t *perm = nullptr;
    const sbn::NItem *geom = nullptr;
    if (pk) {
        if (pk->model != m || pk->bands != b || pk->n_sn != bt->n_sn || pk->n_bands != b->n_bands || pk->device != m->device)
            return SB_EINVAL;
        if (pk->z != bt->z) return SB_EINVAL; // the pack's geometry belongs to the redshift array it was built from
        perm = pk->d_perm;
        geom = reinterpret_cast<const sbn::NItem *>(pk->d_geom);
    } else if (bt->n_sn > 1) {
        const ZWork zw(bt->n_sn);
        unsigned char *ws = scratch_for(b, st, zw.bytes);
        if (!ws) return tl_cuda_err == (int32_t)cudaErrorMemoryAllocation ? SB_ENOMEM : SB_ECUDA;
        const int rc = enqueue_zorder((const float *)bt->z, bt->n_sn, ws, st, &tl_launches);
        if (rc != SB_OK) return rc;
        perm = reinterpret_cast<const int32_t *>(ws + zw.perm_off);
    }
    sbn::SbNParams np;
    memset(&np, 0, sizeof(np));
    np.mp = m->prm;
    np.mx = m->mx_f32;
    np.n_bands = b->n_bands;
    np.n_band_total = b->n_total;
    np.band_off = b->d_off;
    np.band_lam_first = b->d_lam_first;
    np.band_zpab_inv = b->d_zpab_inv;
    np.band_h = b->d_h;
    np.band_dlam = b->d_dlam_f64;
    np.band_w = b->d_w_f32;
    np.band_wd = b->d_wd_f32;
    np.n_sn = bt->n_sn;
    np.n_samples = bt->n_samples;
    np.obs_offset = bt->obs_offset;
    np.time = (const float *)bt->time;
    np.zp = (const float *)bt->zp;
    np.z = (const float *)bt->z;
    np.x0 = (const float *)bt->x0;
    np.x1 = (const float *)bt->x1;
    np.c = (const float *)bt->c;
    np.t0 = (const float *)bt->t0;
    np.band = bt->band;
    np.flux = (const float *)flux;
    np.fluxerr = (const float *)fluxerr;
    np.out_flux = (float *)out_flux;
    np.out_chi2 = (float *)out_chi2;
    np.out_dflux = (float *)out_dflux;
    np.out_dchi2 = (float *)out_dchi2;
    np.perm = perm;
    np.geom = geom;
    np.live = lv.live;
    np.n_live = lv.n_live;
    np.n_groups = (int32_t)n_groups;
    np.cap = cap;
    const int grid = (int)(n_groups < (long long)n_cta ? n_groups : (long long)n_cta);
    const bool small_cl = m->prm.n_cl <= 5;
    if (nu) {
        if (grad) return small_cl ? launch_nw_inst<5, true, true>(m, np, smem, grid, st) : launch_nw_inst<SB_MAX_CL, true, true>(m, np, smem, grid, st);
        return small_cl ? launch_nw_inst<5, false, true>(m, np, smem, grid, st) : launch_nw_inst<SB_MAX_CL, false, true>(m, np, smem, grid, st);
    }
    if (grad) return small_cl ? launch_nw_inst<5, true, false>(m, np, smem, grid, st) : launch_nw_inst<SB_MAX_CL, true, false>(m, np, smem, grid, st);
    return small_cl ? launch_nw_inst<5, false, false>(m, np, smem, grid, st) : launch_nw_inst<SB_MAX_CL, false, false>(m, np, smem, grid, st);
}

int run(const sb_model *m, const sb_bands *b, const sb_batch *bt_in, const void *flux, const void *fluxerr,
        void *out_flux, void *out_dflux, void *out_chi2, void *out_dchi2, void *stream, bool grad,
        const RunLive &lv = RunLive())
{
    tl_launches = 0;
    tl_form = 0;
    if (!m || !b || !bt_in) return SB_EINVAL;
    sb_batch batch = *bt_in; // split the formulation bits off the dtype
    constexpr int32_t kForms = SB_FORM_DIRECT | SB_FORM_GROUPED | SB_FORM_TILED;
    const int32_t form = batch.dtype & kForms;
    batch.dtype &= ~kForms;
    const sb_batch *bt = &batch;
    if (form & (form - 1)) return SB_EINVAL; // at most one formulation bit
    if (bt->dtype != SB_F32 && bt->dtype != SB_F64) return SB_EINVAL;
    if (bt->n_sn < 0 || bt->n_samples < 1 || bt->n_obs_total < 0) return SB_EINVAL;
    if ((out_chi2 || out_dchi2) && (!flux || !fluxerr)) return SB_EINVAL;
    if (bt->n_sn == 0) return SB_OK;
    if (!bt->obs_offset || !bt->z || !bt->x0 || !bt->x1 || !bt->c || !bt->t0) return SB_EINVAL;
    if (bt->n_obs_total > 0 && (!bt->time || !bt->band)) return SB_EINVAL;
    if (!out_flux && !out_dflux && !out_chi2 && !out_dchi2) return SB_EINVAL;
    if ((long long)bt->n_sn * bt->n_samples >= (1LL << 31)) return SB_ELIMIT;
    // the [.][4] gradient outputs are written as 16-byte vectors
    if (((uintptr_t)out_dflux | (uintptr_t)out_dchi2) & (bt->dtype == SB_F32 ? 15u : 31u)) return SB_EINVAL;
    int dev = -1;
    if (!cuda_ok(cudaGetDevice(&dev))) return SB_ECUDA;
    if (dev != m->device || dev != b->device) return SB_EINVAL; // handles live on the device they were loaded on

    SbKParams kp;
    memset(&kp, 0, sizeof(kp));
    kp.mp = m->prm;
    const bool f32 = bt->dtype == SB_F32;
    kp.m0 = f32 ? (const void *)m->m0_f32 : (const void *)m->m0_f64;
    kp.m1 = f32 ? (const void *)m->m1_f32 : (const void *)m->m1_f64;
    kp.n_bands = b->n_bands;
    kp.n_band_total = b->n_total;
    kp.band_off = b->d_off;
    kp.band_lam_first = b->d_lam_first;
    kp.band_zpab_inv = b->d_zpab_inv;
    kp.band_tab = f32 ? (const void *)b->d_tab_f32 : (const void *)b->d_tab_f64;
    kp.n_sn = bt->n_sn;
    kp.n_samples = bt->n_samples;
    kp.obs_offset = bt->obs_offset;
    kp.time = bt->time;
    kp.zp = bt->zp;
    kp.z = bt->z;
    kp.x0 = bt->x0;
    kp.x1 = bt->x1;
    kp.c = bt->c;
    kp.t0 = bt->t0;
    kp.band = bt->band;
    kp.flux = flux;
    kp.fluxerr = fluxerr;
    kp.out_flux = out_flux;
    kp.out_dflux = out_dflux;
    kp.out_chi2 = out_chi2;
    kp.out_dchi2 = out_dchi2;
    kp.n_live = lv.n_live;
    cudaStream_t st = (cudaStream_t)stream;
    // automatic choice: calls too small to fill the warps of one CTA per SM go to the direct kernel
    const bool tiny = form == 0 && (long long)bt->n_obs_total * bt->n_samples < 4096;
    if (f32 && form != SB_FORM_DIRECT && !tiny && bt->n_obs_total > 0) {
        if (form != SB_FORM_GROUPED) {
            const int rc = launch_nw(grad, m, b, bt, flux, fluxerr, out_flux, out_chi2, out_dflux, out_dchi2, st, lv);
            if (rc != 1) return rc;
        }
        if (form != SB_FORM_TILED && !grad) {
            const int rc = launch_hoist(m, b, bt, flux, fluxerr, out_flux, out_chi2, st);
            if (rc != 1) return rc;
        }
    }
    if (form == SB_FORM_GROUPED || form == SB_FORM_TILED) return SB_ELIMIT; // demanded but does not apply
    if (f32) {
        if (grad) return launch_typed<float, true, 8>(m, kp, b, bt->n_obs_total, st);
        return launch_typed<float, false, 16>(m, kp, b, bt->n_obs_total, st);
    }
    if (grad) return launch_typed<double, true, 8>(m, kp, b, bt->n_obs_total, st);
    return launch_typed<double, false, 8>(m, kp, b, bt->n_obs_total, st);
}

} // namespace

extern "C" {

int sb_pack_observations(const sb_model *m, const sb_bands *b, const sb_batch *bt, void *stream, sb_pack **out)
{
    NvtxRange nvtx("sb_pack_observations");
    if (out) *out = nullptr;
    if (!m || !b || !bt || !out) return SB_EINVAL;
    if ((bt->dtype & 0xff) != SB_F32 || bt->n_sn < 1 || !bt->z) return SB_EINVAL;
    if (b->n_bands > sbn::kMaxBands) return SB_ELIMIT; // the kernel that uses a pack does not apply
    int dev = -1;
    if (!cuda_ok(cudaGetDevice(&dev))) return SB_ECUDA;
    if (dev != m->device || dev != b->device) return SB_EINVAL;
    sb_pack *h = new (std::nothrow) sb_pack();
    if (!h) return SB_ENOMEM;
    memset(h, 0, sizeof(*h));
    h->n_sn = bt->n_sn;
    h->n_bands = b->n_bands;
    h->model = m;
    h->bands = b;
    h->z = bt->z;
    h->device = dev;
    const ZWork zw(bt->n_sn);
    const size_t geom_bytes = sizeof(sbn::NItem) * (size_t)bt->n_sn * b->n_bands;
    if (!cuda_ok(cudaMalloc((void **)&h->d_ws, zw.bytes)) || !cuda_ok(cudaMalloc(&h->d_geom, geom_bytes))) {
        const int rc = tl_cuda_err == (int32_t)cudaErrorMemoryAllocation ? SB_ENOMEM : SB_ECUDA;
        sb_free_pack(h);
        return rc;
    }
    h->d_perm = reinterpret_cast<int32_t *>(h->d_ws + zw.perm_off);
    cudaStream_t st = (cudaStream_t)stream;
    int32_t launches = 0;
    int rc = enqueue_zorder((const float *)bt->z, bt->n_sn, h->d_ws, st, &launches);
    if (rc == SB_OK) {
        const long long n_items = (long long)bt->n_sn * b->n_bands;
        const sbn::NBandsView bv{b->n_bands, b->all_uniform, b->d_off, b->d_lam_first, b->d_h, b->d_dlam_f64};
        sbn::sb_geom_kernel<<<(unsigned)((n_items + 255) / 256), 256, 0, st>>>(m->prm, bv, (const float *)bt->z, bt->n_sn,
                                                                             reinterpret_cast<sbn::NItem *>(h->d_geom));
        if (!cuda_ok(cudaGetLastError())) rc = SB_ECUDA;
        else launches += 1;
    }
    if (rc != SB_OK) { sb_free_pack(h); return rc; }
    tl_launches = launches;
    *out = h;
    return SB_OK;
}

void sb_free_pack(sb_pack *p)
{
    if (!p) return;
    cudaFree(p->d_ws);
    cudaFree(p->d_geom);
    delete p;
}

int sb_bandflux(const sb_model *m, const sb_bands *b, const sb_batch *batch, void *out_flux, void *stream)
{
    NvtxRange nvtx("sb_bandflux");
    if (!out_flux && !(batch && batch->n_sn == 0)) { tl_launches = 0; return SB_EINVAL; }
    return run(m, b, batch, nullptr, nullptr, out_flux, nullptr, nullptr, nullptr, stream, false);
}

int sb_chi2(const sb_model *m, const sb_bands *b, const sb_batch *batch, const void *flux, const void *fluxerr,
            void *out_chi2, void *out_flux, void *stream)
{
    NvtxRange nvtx("sb_chi2");
    if ((!out_chi2 || !flux || !fluxerr) && !(batch && batch->n_sn == 0)) { tl_launches = 0; return SB_EINVAL; }
    return run(m, b, batch, flux, fluxerr, out_flux, nullptr, out_chi2, nullptr, stream, false);
}

} // extern "C"

// ---------------------------------------------------------------- sb_chi2_noalloc
// Scratch of the allocation-free chi^2 call: the z-order workspace (ZWork layout) of a batch of up to
// SB_NOALLOC_MAX_SN supernovae, as a fixed array in the library image.  Each GPU that loads the library holds
// its own copy until the process exits.  In HOST code the name below is only a handle for the runtime -- it is
// not a device address and must never be handed to a kernel or to cudaMemsetAsync; noalloc_scratch() asks the
// runtime for the real address on the current device.
constexpr size_t kNoAllocBytes = 4096 + (((sizeof(int32_t) * (size_t)SB_NOALLOC_MAX_SN) + 255) & ~(size_t)255) +
                                 sizeof(uint32_t) * (size_t)sbh::kZSegs * sbh::kZBins;
static __device__ __align__(256) unsigned char sb_noalloc_scratch[kNoAllocBytes];

namespace {

// Device address of sb_noalloc_scratch on `device`, which must be the current device.  Looked up once per
// device (cudaGetSymbolAddress; the first lookup also makes the runtime load this module on that device) and
// cached; NULL on failure, with the CUDA error left in tl_cuda_err.
unsigned char *noalloc_scratch(int device)
{
    constexpr int kMaxDev = 64;
    static std::mutex mu;
    static unsigned char *addr[kMaxDev] = {};
    if (device < 0 || device >= kMaxDev) { tl_cuda_err = (int32_t)cudaErrorInvalidDevice; return nullptr; }
    std::lock_guard<std::mutex> lock(mu);
    if (!addr[device]) {
        void *p = nullptr;
        if (!cuda_ok(cudaGetSymbolAddress(&p, sb_noalloc_scratch)) || !p) return nullptr;
        addr[device] = static_cast<unsigned char *>(p);
    }
    return addr[device];
}

} // namespace

extern "C" {

int sb_chi2_noalloc(const sb_model *m, const sb_bands *b, const sb_batch *batch, const void *flux,
                    const void *fluxerr, void *out_chi2, void *out_flux, void *stream)
{
    NvtxRange nvtx("sb_chi2_noalloc");
    tl_launches = 0;
    tl_form = 0;
    if (!m || !b || !batch) return SB_EINVAL;
    // the size limit of the fixed array comes first: refused before anything else is looked at or enqueued
    if (batch->n_sn > SB_NOALLOC_MAX_SN) return SB_ELIMIT;
    if ((!out_chi2 || !flux || !fluxerr) && batch->n_sn != 0) return SB_EINVAL;
    if (batch->pack) return SB_EINVAL; // with a pack sb_chi2 itself allocates nothing
    constexpr int32_t kForms = SB_FORM_DIRECT | SB_FORM_GROUPED | SB_FORM_TILED;
    const int32_t form = batch->dtype & kForms;
    if ((batch->dtype & ~kForms) != SB_F32 || (form != 0 && form != SB_FORM_TILED)) return SB_EINVAL;
    if (batch->n_sn < 0) return SB_EINVAL;
    if (ZWork(batch->n_sn).bytes > kNoAllocBytes) return SB_ELIMIT; // cannot happen while the layouts agree
    int dev = -1;
    if (!cuda_ok(cudaGetDevice(&dev))) return SB_ECUDA;
    if (dev != m->device || dev != b->device) return SB_EINVAL;
    unsigned char *ws = noalloc_scratch(dev);
    if (!ws) return SB_ECUDA;
    // Run the unchanged sb_chi2 path with the fixed array standing where a pack's redshift order stands: the
    // permutation is rebuilt into the array by this call (enqueue_zorder clears the counters it needs at zero
    // and overwrites the rest), there is no item geometry (d_geom NULL: the kernel computes it, as it does
    // without a pack), and SB_FORM_TILED makes run() return SB_ELIMIT rather than fall through to a kernel
    // that would take a workspace from scratch_for().  A single supernova needs no order at all.
    // Batches too small for that kernel (the same threshold as sb_chi2's own choice) go to the direct kernel,
    // which uses no scratch.
    sb_pack view;
    memset(&view, 0, sizeof(view));
    sb_batch bt = *batch;
    const bool tiny = (long long)bt.n_obs_total * bt.n_samples < 4096;
    bt.dtype = SB_F32 | (tiny ? SB_FORM_DIRECT : SB_FORM_TILED);
    int32_t sort_launches = 0;
    if (bt.n_sn > 1 && !tiny) {
        if (!bt.z) return SB_EINVAL;
        view.n_sn = bt.n_sn;
        view.n_bands = b->n_bands;
        view.model = m;
        view.bands = b;
        view.z = bt.z;
        view.device = dev;
        view.d_perm = reinterpret_cast<int32_t *>(ws + ZWork(bt.n_sn).perm_off);
        const int rc = enqueue_zorder((const float *)bt.z, bt.n_sn, ws, (cudaStream_t)stream, &sort_launches);
        if (rc != SB_OK) return rc;
        bt.pack = &view;
    }
    const int rc = run(m, b, &bt, flux, fluxerr, out_flux, nullptr, out_chi2, nullptr, stream, false);
    if (rc == SB_OK) tl_launches += sort_launches;
    return rc;
}

int sb_bandflux_grad(const sb_model *m, const sb_bands *b, const sb_batch *batch, const void *flux,
                     const void *fluxerr, void *out_flux, void *out_dflux, void *out_chi2, void *out_dchi2,
                     void *stream)
{
    NvtxRange nvtx("sb_bandflux_grad");
    return run(m, b, batch, flux, fluxerr, out_flux, out_dflux, out_chi2, out_dchi2, stream, true);
}

} // extern "C"

// ------------------------------------------------------------------------------------------
// Host-buffer entry points: chunked staging with copy / compute overlap
// ------------------------------------------------------------------------------------------
namespace {

constexpr int kHostStreams = 3;

struct ChunkBufs {
    int32_t *obs_offset = nullptr, *band = nullptr;
    unsigned char *time = nullptr, *zp = nullptr, *flux = nullptr, *fluxerr = nullptr;
    unsigned char *z = nullptr, *x0 = nullptr, *x1 = nullptr, *c = nullptr, *t0 = nullptr;
    unsigned char *o_flux = nullptr, *o_dflux = nullptr, *o_chi2 = nullptr, *o_dchi2 = nullptr;
};

int run_host(const sb_model *m, const sb_bands *b, const sb_batch *hb, const void *flux, const void *fluxerr,
             void *out_flux, void *out_dflux, void *out_chi2, void *out_dchi2, bool grad)
{
    tl_launches = 0;
    tl_form = 0;
    if (!m || !b || !hb) return SB_EINVAL;
    const int32_t base_dtype = hb->dtype & 0xff;
    if (base_dtype != SB_F32 && base_dtype != SB_F64) return SB_EINVAL;
    if (hb->n_sn < 0 || hb->n_samples < 1 || hb->n_obs_total < 0) return SB_EINVAL;
    if ((out_chi2 || out_dchi2) && (!flux || !fluxerr)) return SB_EINVAL;
    if (!out_flux && !out_dflux && !out_chi2 && !out_dchi2) return SB_EINVAL;
    if (hb->n_sn == 0) return SB_OK;
    if (!hb->obs_offset || !hb->z || !hb->x0 || !hb->x1 || !hb->c || !hb->t0) return SB_EINVAL;
    if (hb->n_obs_total > 0 && (!hb->time || !hb->band)) return SB_EINVAL;
    if (hb->obs_offset[0] != 0 || hb->obs_offset[hb->n_sn] != hb->n_obs_total) return SB_EINVAL;
    const size_t es = base_dtype == SB_F32 ? 4 : 8;
    const long long ns = hb->n_samples;
    const int n_sm = m->n_sm;
    int dev = -1;
    if (!cuda_ok(cudaGetDevice(&dev))) return SB_ECUDA;
    if (dev != m->device || dev != b->device) return SB_EINVAL;
    if (hb->pack) return SB_EINVAL; // a pack describes the whole device-resident batch, not its chunks

    // chunks of supernovae: about 24 MB of inputs + outputs each, at most 32 chunks, and (one sample per
    // supernova) a multiple of n_sm * 32 supernovae so that every chunk fills whole waves of groups
    const double bytes_per_sn =
        ((double)hb->n_obs_total / hb->n_sn) * (double)((hb->zp ? 3 : 2) * es + 4 + (flux ? 2 * es : 0) +
                                                        (out_flux ? ns * es : 0) + (out_dflux ? 4 * ns * es : 0)) +
        (double)(5 * ns * es);
    long long chunk_sn = (long long)(24.0 * 1024 * 1024 / (bytes_per_sn > 1.0 ? bytes_per_sn : 1.0));
    if (chunk_sn * 32 < hb->n_sn) chunk_sn = (hb->n_sn + 31) / 32;
    const long long wave = (long long)n_sm * 32;
    if (ns == 1 && chunk_sn > wave) chunk_sn = (chunk_sn / wave) * wave;
    if (chunk_sn < 1) chunk_sn = 1;
    if (chunk_sn > hb->n_sn) chunk_sn = hb->n_sn;
    long long max_obs = 0; // observations of the largest chunk
    for (long long s0 = 0; s0 < hb->n_sn; s0 += chunk_sn) {
        const long long s1 = s0 + chunk_sn < hb->n_sn ? s0 + chunk_sn : hb->n_sn;
        const long long n = (long long)hb->obs_offset[s1] - hb->obs_offset[s0];
        if (n < 0) return SB_EINVAL;
        if (n > max_obs) max_obs = n;
    }

    // context of this call: three internal streams and one staging slab per stream, owned by the bands
    // handle, taken from its pool (one context per concurrent host call) and returned before the call ends
    SbScratch *sc = b->scratch;
    SbScratch::HostCtx *ctx = nullptr;
    {
        std::lock_guard<std::mutex> lock(sc->mu);
        for (auto *c : sc->host)
            if (!c->busy) { ctx = c; break; }
        if (!ctx) {
            ctx = new (std::nothrow) SbScratch::HostCtx();
            if (!ctx) return SB_ENOMEM;
            memset(ctx, 0, sizeof(*ctx));
            sc->host.push_back(ctx);
        }
        ctx->busy = true;
    }
    struct Release {
        SbScratch *sc; SbScratch::HostCtx *c;
        ~Release() { std::lock_guard<std::mutex> lock(sc->mu); c->busy = false; }
    } release{sc, ctx};
    int rc = SB_OK;
    for (int i = 0; i < kHostStreams && rc == SB_OK; ++i)
        if (!ctx->st[i] && !cuda_ok(cudaStreamCreateWithFlags(&ctx->st[i], cudaStreamNonBlocking))) rc = SB_ECUDA;
    if (rc != SB_OK) return rc;
    cudaStream_t *st = ctx->st;
    // one slab per stream, carved into the chunk's arrays (256-byte aligned); a free context has no work
    // in flight (every call synchronises its streams before it returns), so its slabs can be regrown
    ChunkBufs bufs[kHostStreams];
    unsigned char **slab = ctx->slab;
    const int n_streams = kHostStreams;
    const size_t mo = (size_t)max_obs, mu = (size_t)(chunk_sn * ns);
    for (int pass = 0; pass < 2 && rc == SB_OK; ++pass) { // pass 0: size, pass 1: carve
        size_t total = 0;
        for (int i = 0; i < (pass == 0 ? 1 : n_streams); ++i) {
            size_t off = 0;
            auto carve = [&](auto &ptr, size_t bytes) {
                if (pass == 1) ptr = reinterpret_cast<std::remove_reference_t<decltype(ptr)>>(slab[i] + off);
                off += (bytes + 255) & ~(size_t)255;
            };
            ChunkBufs &B = bufs[i];
            carve(B.obs_offset, sizeof(int32_t) * (size_t)(chunk_sn + 1));
            carve(B.band, sizeof(int32_t) * mo);
            carve(B.time, es * mo);
            if (hb->zp) carve(B.zp, es * mo);
            if (flux) { carve(B.flux, es * mo); carve(B.fluxerr, es * mo); }
            carve(B.z, es * (size_t)chunk_sn);
            carve(B.x0, es * mu); carve(B.x1, es * mu); carve(B.c, es * mu); carve(B.t0, es * mu);
            if (out_flux) carve(B.o_flux, es * mo * (size_t)ns);
            if (out_dflux) carve(B.o_dflux, 4 * es * mo * (size_t)ns);
            if (out_chi2) carve(B.o_chi2, es * mu);
            if (out_dchi2) carve(B.o_dchi2, 4 * es * mu);
            total = off;
        }
        if (pass == 0 && total > ctx->slab_bytes) {
            for (int i = 0; i < n_streams; ++i) {
                if (slab[i]) cudaFree(slab[i]);
                slab[i] = nullptr;
            }
            ctx->slab_bytes = 0;
            for (int i = 0; i < n_streams && rc == SB_OK; ++i)
                if (!cuda_ok(cudaMalloc((void **)&slab[i], total)))
                    rc = tl_cuda_err == (int32_t)cudaErrorMemoryAllocation ? SB_ENOMEM : SB_ECUDA;
            if (rc == SB_OK) ctx->slab_bytes = total;
        }
    }
    int32_t launches = 0, form = 0;
    int k = 0;
    for (long long s0 = 0; s0 < hb->n_sn && rc == SB_OK; s0 += chunk_sn, ++k) {
        const long long s1 = s0 + chunk_sn < hb->n_sn ? s0 + chunk_sn : hb->n_sn;
        const long long o0 = hb->obs_offset[s0], o1 = hb->obs_offset[s1];
        const size_t nsn = (size_t)(s1 - s0), nob = (size_t)(o1 - o0), nun = nsn * (size_t)ns;
        cudaStream_t s = st[k % kHostStreams];
        ChunkBufs &B = bufs[k % kHostStreams];
        auto h2d = [&](void *dst, const void *src, size_t off, size_t bytes) {
            if (rc == SB_OK && bytes && !cuda_ok(cudaMemcpyAsync(dst, (const unsigned char *)src + off, bytes, cudaMemcpyHostToDevice, s)))
                rc = SB_ECUDA;
        };
        auto d2h = [&](void *dst, size_t off, const void *src, size_t bytes) {
            if (rc == SB_OK && bytes && !cuda_ok(cudaMemcpyAsync((unsigned char *)dst + off, src, bytes, cudaMemcpyDeviceToHost, s)))
                rc = SB_ECUDA;
        };
        h2d(B.obs_offset, hb->obs_offset, sizeof(int32_t) * (size_t)s0, sizeof(int32_t) * (nsn + 1));
        h2d(B.band, hb->band, sizeof(int32_t) * (size_t)o0, sizeof(int32_t) * nob);
        h2d(B.time, hb->time, es * (size_t)o0, es * nob);
        if (hb->zp) h2d(B.zp, hb->zp, es * (size_t)o0, es * nob);
        if (flux) { h2d(B.flux, flux, es * (size_t)o0, es * nob); h2d(B.fluxerr, fluxerr, es * (size_t)o0, es * nob); }
        h2d(B.z, hb->z, es * (size_t)s0, es * nsn);
        h2d(B.x0, hb->x0, es * (size_t)(s0 * ns), es * nun);
        h2d(B.x1, hb->x1, es * (size_t)(s0 * ns), es * nun);
        h2d(B.c, hb->c, es * (size_t)(s0 * ns), es * nun);
        h2d(B.t0, hb->t0, es * (size_t)(s0 * ns), es * nun);
        if (rc != SB_OK) break;
        // the chunk keeps the caller's (absolute) observation offsets: per-observation device arrays are
        // addressed through pointers shifted back by the chunk's first observation
        sb_batch cb = *hb;
        cb.n_sn = (int32_t)nsn;
        cb.n_obs_total = (int32_t)nob;
        cb.obs_offset = B.obs_offset;
        cb.band = B.band - o0;
        cb.time = B.time - es * (size_t)o0;
        cb.zp = hb->zp ? B.zp - es * (size_t)o0 : nullptr;
        cb.z = B.z; cb.x0 = B.x0; cb.x1 = B.x1; cb.c = B.c; cb.t0 = B.t0;
        const void *d_flux = flux ? B.flux - es * (size_t)o0 : nullptr;
        const void *d_err = flux ? B.fluxerr - es * (size_t)o0 : nullptr;
        void *d_oflux = out_flux ? B.o_flux - es * (size_t)(o0 * ns) : nullptr;
        void *d_odflux = out_dflux ? B.o_dflux - 4 * es * (size_t)(o0 * ns) : nullptr;
        rc = run(m, b, &cb, d_flux, d_err, d_oflux, d_odflux, B.o_chi2, B.o_dchi2, (void *)s, grad);
        launches += tl_launches;
        if (tl_form) form = tl_form;
        if (rc != SB_OK) break;
        if (out_flux) d2h(out_flux, es * (size_t)(o0 * ns), B.o_flux, es * nob * (size_t)ns);
        if (out_dflux) d2h(out_dflux, 4 * es * (size_t)(o0 * ns), B.o_dflux, 4 * es * nob * (size_t)ns);
        if (out_chi2) d2h(out_chi2, es * (size_t)(s0 * ns), B.o_chi2, es * nun);
        if (out_dchi2) d2h(out_dchi2, 4 * es * (size_t)(s0 * ns), B.o_dchi2, 4 * es * nun);
    }
    for (int i = 0; i < n_streams; ++i)
        if (!cuda_ok(cudaStreamSynchronize(st[i])) && rc == SB_OK) rc = SB_ECUDA;
    tl_launches = rc == SB_OK ? launches : 0;
    tl_form = rc == SB_OK ? form : 0;
    return rc;
}

} // namespace

extern "C" {

int sb_chi2_host(const sb_model *m, const sb_bands *b, const sb_batch *batch, const void *flux, const void *fluxerr,
                 void *out_chi2, void *out_flux)
{
    NvtxRange nvtx("sb_chi2_host");
    if ((!out_chi2 || !flux || !fluxerr) && !(batch && batch->n_sn == 0)) { tl_launches = 0; return SB_EINVAL; }
    return run_host(m, b, batch, flux, fluxerr, out_flux, nullptr, out_chi2, nullptr, false);
}

int sb_bandflux_grad_host(const sb_model *m, const sb_bands *b, const sb_batch *batch, const void *flux,
                          const void *fluxerr, void *out_flux, void *out_dflux, void *out_chi2, void *out_dchi2)
{
    return run_host(m, b, batch, flux, fluxerr, out_flux, out_dflux, out_chi2, out_dchi2, true);
}

} // extern "C"

// ------------------------------------------------------------------------------------------
// Device-resident batched L-BFGS fit (sb_fit.cuh): one lane per unit, no host synchronisation
// ------------------------------------------------------------------------------------------
namespace {

constexpr double kFtolFloorF32 = 4.76837158203125e-7; // 2^-21 = 8 fp32 ulps of chi^2 (include/saltband.h: sb_fit_lbfgs)

struct FitLayout { // carve-up of the fit workspace (kScratchFit slot of the call's stream)
    size_t theta[4], chi2, dchi2, u, g, d, ut, f, alpha, scale, S, Y, ints[7], n_live, bytes;
    FitLayout(size_t n, size_t es, int memory)
    {
        size_t o = 0;
        auto take = [&](size_t b) { const size_t at = o; o += (b + 255) & ~(size_t)255; return at; };
        for (int k = 0; k < 4; ++k) theta[k] = take(es * n);
        chi2 = take(es * n);
        dchi2 = take(4 * es * n);
        u = take(32 * n); g = take(32 * n); d = take(32 * n); ut = take(32 * n);
        f = take(8 * n); alpha = take(8 * n); scale = take(8 * n);
        S = take((size_t)memory * 32 * n); Y = take((size_t)memory * 32 * n);
        for (int k = 0; k < 7; ++k) ints[k] = take(4 * n);
        n_live = take(256);
        bytes = o;
    }
};

int fit_check_opts(const sb_fit_opts *o)
{
    if (!o) return SB_EINVAL;
    if (o->memory < 1 || o->memory > sbf::kMaxMemory || o->max_eval < 1 || o->max_iter < 1 || o->trace_len < 0) return SB_EINVAL;
    if (!(o->ftol >= 0.0) || !(o->gtol >= 0.0)) return SB_EINVAL;
    if (o->lo && o->hi)
        for (int k = 0; k < 4; ++k)
            if (!(o->lo[k] <= o->hi[k])) return SB_EINVAL;
    return SB_OK;
}

int fit_device(const sb_model *m, const sb_bands *b, const sb_batch *bt_in, const void *flux, const void *fluxerr,
               const sb_fit_opts *opts, const sb_fit_result *res, cudaStream_t st)
{
    tl_launches = 0;
    tl_form = 0;
    if (!m || !b || !bt_in || !flux || !fluxerr || !res) return SB_EINVAL;
    int rc = fit_check_opts(opts);
    if (rc != SB_OK) return rc;
    const int32_t base = bt_in->dtype & 0xff;
    if (base != SB_F32 && base != SB_F64) return SB_EINVAL;
    if (bt_in->n_sn < 0 || bt_in->n_samples < 1 || bt_in->n_obs_total < 0) return SB_EINVAL;
    if (bt_in->n_sn == 0) return SB_OK;
    if (!res->theta || !res->chi2) return SB_EINVAL;
    if (opts->trace_len > 0 && !res->trace) return SB_EINVAL;
    if (!bt_in->x0 || !bt_in->x1 || !bt_in->c || !bt_in->t0) return SB_EINVAL;
    const long long n_units = (long long)bt_in->n_sn * bt_in->n_samples;
    if (n_units >= (1LL << 31)) return SB_ELIMIT;
    int dev = -1;
    if (!cuda_ok(cudaGetDevice(&dev))) return SB_ECUDA;
    if (dev != m->device || dev != b->device) return SB_EINVAL;
    const size_t es = base == SB_F32 ? 4 : 8, n = (size_t)n_units;
    const FitLayout L(n, es, opts->memory);
    unsigned char *ws = scratch_for(b, st, L.bytes, kScratchFit);
    if (!ws) return tl_cuda_err == (int32_t)cudaErrorMemoryAllocation ? SB_ENOMEM : SB_ECUDA;

    sbf::FitParams F;
    memset(&F, 0, sizeof(F));
    F.st.u = (double *)(ws + L.u); F.st.g = (double *)(ws + L.g); F.st.d = (double *)(ws + L.d); F.st.ut = (double *)(ws + L.ut);
    F.st.f = (double *)(ws + L.f); F.st.alpha = (double *)(ws + L.alpha); F.st.scale = (double *)(ws + L.scale);
    F.st.S = (double *)(ws + L.S); F.st.Y = (double *)(ws + L.Y);
    F.st.n_hist = (int32_t *)(ws + L.ints[0]); F.st.head = (int32_t *)(ws + L.ints[1]); F.st.n_eval = (int32_t *)(ws + L.ints[2]);
    F.st.n_iter = (int32_t *)(ws + L.ints[3]); F.st.n_back = (int32_t *)(ws + L.ints[4]); F.st.status = (int32_t *)(ws + L.ints[5]);
    F.st.live = (int32_t *)(ws + L.ints[6]);
    F.st.n_live = (int32_t *)(ws + L.n_live);
    F.n = (int32_t)n_units;
    F.memory = opts->memory; F.max_eval = opts->max_eval; F.max_iter = opts->max_iter; F.trace_len = opts->trace_len;
    F.ftol = opts->ftol; F.gtol = opts->gtol;
    // SB_F32: chi^2 comes back from the kernels in fp32, so a decrease of less than a few of its ulps cannot be
    // observed; a positive ftol below that resolution would never be met before the line search stalls
    if (base == SB_F32 && F.ftol > 0.0 && F.ftol < kFtolFloorF32) F.ftol = kFtolFloorF32;
    F.has_box = (opts->lo || opts->hi) ? 1 : 0;
    for (int k = 0; k < 4; ++k) {
        F.lo[k] = opts->lo ? opts->lo[k] : -INFINITY;
        F.hi[k] = opts->hi ? opts->hi[k] : INFINITY;
    }
    F.x0 = ws + L.theta[0]; F.x1 = ws + L.theta[1]; F.c = ws + L.theta[2]; F.t0 = ws + L.theta[3];
    F.chi2 = ws + L.chi2; F.dchi2 = ws + L.dchi2;
    F.theta_out = res->theta; F.chi2_out = res->chi2;
    F.status_out = res->status; F.n_iter_out = res->n_iter; F.n_eval_out = res->n_eval;
    F.trace_out = res->trace;

    const unsigned blocks_i = (unsigned)((n + 255) / 256), blocks_u = (unsigned)((n + 127) / 128);
    int32_t launches = 0, form = 0;
    if (base == SB_F32)
        sbf::sb_fit_init_kernel<float><<<blocks_i, 256, 0, st>>>(F, (const float *)bt_in->x0, (const float *)bt_in->x1,
                                                                  (const float *)bt_in->c, (const float *)bt_in->t0);
    else
        sbf::sb_fit_init_kernel<double><<<blocks_i, 256, 0, st>>>(F, (const double *)bt_in->x0, (const double *)bt_in->x1,
                                                                   (const double *)bt_in->c, (const double *)bt_in->t0);
    if (!cuda_ok(cudaGetLastError())) return SB_ECUDA;
    launches += 1;
    sb_batch eb = *bt_in; // the evaluation batch: the caller's observations at the lanes' trial parameters
    eb.x0 = F.x0; eb.x1 = F.x1; eb.c = F.c; eb.t0 = F.t0;
    const RunLive lv{F.st.live, F.st.n_live};
    for (int e = 0; e < opts->max_eval; ++e) {
        rc = run(m, b, &eb, flux, fluxerr, nullptr, nullptr, ws + L.chi2, ws + L.dchi2, (void *)st, true, lv);
        if (rc != SB_OK) return rc;
        launches += tl_launches;
        form = tl_form;
        if (base == SB_F32) sbf::sb_fit_update_kernel<float><<<blocks_u, 128, 0, st>>>(F);
        else sbf::sb_fit_update_kernel<double><<<blocks_u, 128, 0, st>>>(F);
        if (!cuda_ok(cudaGetLastError())) return SB_ECUDA;
        launches += 1;
    }
    tl_launches = launches;
    tl_form = form;
    return SB_OK;
}

} // namespace

extern "C" {

void sb_fit_default_opts(sb_fit_opts *o)
{
    if (!o) return;
    o->memory = 8;
    o->max_eval = 60;
    o->max_iter = 1000;
    o->trace_len = 0;
    o->ftol = 1e-12;
    o->gtol = 0.0;
    o->lo = nullptr;
    o->hi = nullptr;
}

int sb_fit_lbfgs(const sb_model *m, const sb_bands *b, const sb_batch *batch, const void *flux, const void *fluxerr,
                 const sb_fit_opts *opts, const sb_fit_result *result, void *stream)
{
    NvtxRange nvtx("sb_fit_lbfgs");
    return fit_device(m, b, batch, flux, fluxerr, opts, result, (cudaStream_t)stream);
}

int sb_fit_lbfgs_host(const sb_model *m, const sb_bands *b, const sb_batch *hb, const void *flux, const void *fluxerr,
                      const sb_fit_opts *opts, const sb_fit_result *hres)
{
    NvtxRange nvtx("sb_fit_lbfgs_host");
    tl_launches = 0;
    tl_form = 0;
    if (!m || !b || !hb || !flux || !fluxerr || !hres) return SB_EINVAL;
    int rc = fit_check_opts(opts);
    if (rc != SB_OK) return rc;
    const int32_t base = hb->dtype & 0xff;
    if (base != SB_F32 && base != SB_F64) return SB_EINVAL;
    if (hb->n_sn < 0 || hb->n_samples < 1 || hb->n_obs_total < 0 || hb->pack) return SB_EINVAL;
    if (hb->n_sn == 0) return SB_OK;
    if (!hb->obs_offset || !hb->z || !hb->x0 || !hb->x1 || !hb->c || !hb->t0 || !hres->theta || !hres->chi2) return SB_EINVAL;
    if (hb->n_obs_total > 0 && (!hb->time || !hb->band)) return SB_EINVAL;
    if (hb->obs_offset[0] != 0 || hb->obs_offset[hb->n_sn] != hb->n_obs_total) return SB_EINVAL;
    if (opts->trace_len > 0 && !hres->trace) return SB_EINVAL;
    int dev = -1;
    if (!cuda_ok(cudaGetDevice(&dev))) return SB_ECUDA;
    if (dev != m->device || dev != b->device) return SB_EINVAL;
    const size_t es = base == SB_F32 ? 4 : 8;
    const size_t nsn = (size_t)hb->n_sn, nob = (size_t)hb->n_obs_total, nun = nsn * (size_t)hb->n_samples;

    // the whole batch stays resident for the fit: one staging slab of a host-call context of the handle
    SbScratch *sc = b->scratch;
    SbScratch::HostCtx *ctx = nullptr;
    {
        std::lock_guard<std::mutex> lock(sc->mu);
        for (auto *c : sc->host)
            if (!c->busy) { ctx = c; break; }
        if (!ctx) {
            ctx = new (std::nothrow) SbScratch::HostCtx();
            if (!ctx) return SB_ENOMEM;
            memset(ctx, 0, sizeof(*ctx));
            sc->host.push_back(ctx);
        }
        ctx->busy = true;
    }
    struct Release {
        SbScratch *sc; SbScratch::HostCtx *c;
        ~Release() { std::lock_guard<std::mutex> lock(sc->mu); c->busy = false; }
    } release{sc, ctx};
    if (!ctx->st[0] && !cuda_ok(cudaStreamCreateWithFlags(&ctx->st[0], cudaStreamNonBlocking))) return SB_ECUDA;
    cudaStream_t st = ctx->st[0];
    size_t off = 0;
    auto take = [&](size_t bytes) { const size_t at = off; off += (bytes + 255) & ~(size_t)255; return at; };
    const size_t o_off = take(4 * (nsn + 1)), o_band = take(4 * nob), o_time = take(es * nob), o_zp = take(hb->zp ? es * nob : 0),
                 o_flux = take(es * nob), o_err = take(es * nob), o_z = take(es * nsn), o_x0 = take(es * nun), o_x1 = take(es * nun),
                 o_c = take(es * nun), o_t0 = take(es * nun), r_theta = take(4 * es * nun), r_chi2 = take(es * nun),
                 r_status = take(4 * nun), r_iter = take(4 * nun), r_eval = take(4 * nun),
                 r_trace = take(8 * (size_t)opts->trace_len * nun);
    if (off > ctx->fit_bytes) { // a free context has no work in flight: its slab can be regrown
        if (ctx->fit_slab) cudaFree(ctx->fit_slab);
        ctx->fit_slab = nullptr;
        ctx->fit_bytes = 0;
        if (!cuda_ok(cudaMalloc((void **)&ctx->fit_slab, off)))
            return tl_cuda_err == (int32_t)cudaErrorMemoryAllocation ? SB_ENOMEM : SB_ECUDA;
        ctx->fit_bytes = off;
    }
    unsigned char *D = ctx->fit_slab;
    rc = SB_OK;
    auto h2d = [&](size_t at, const void *src, size_t bytes) {
        if (rc == SB_OK && bytes && !cuda_ok(cudaMemcpyAsync(D + at, src, bytes, cudaMemcpyHostToDevice, st))) rc = SB_ECUDA;
    };
    auto d2h = [&](void *dst, size_t at, size_t bytes) {
        if (rc == SB_OK && dst && bytes && !cuda_ok(cudaMemcpyAsync(dst, D + at, bytes, cudaMemcpyDeviceToHost, st))) rc = SB_ECUDA;
    };
    h2d(o_off, hb->obs_offset, 4 * (nsn + 1)); h2d(o_band, hb->band, 4 * nob); h2d(o_time, hb->time, es * nob);
    if (hb->zp) h2d(o_zp, hb->zp, es * nob);
    h2d(o_flux, flux, es * nob); h2d(o_err, fluxerr, es * nob); h2d(o_z, hb->z, es * nsn);
    h2d(o_x0, hb->x0, es * nun); h2d(o_x1, hb->x1, es * nun); h2d(o_c, hb->c, es * nun); h2d(o_t0, hb->t0, es * nun);
    if (rc != SB_OK) { // copies enqueued before the failing one may still read the caller's buffers: drain first
        cudaStreamSynchronize(st);
        return rc;
    }
    sb_batch db = *hb;
    db.obs_offset = (const int32_t *)(D + o_off); db.band = (const int32_t *)(D + o_band); db.time = D + o_time;
    db.zp = hb->zp ? D + o_zp : nullptr; db.z = D + o_z; db.x0 = D + o_x0; db.x1 = D + o_x1; db.c = D + o_c; db.t0 = D + o_t0;
    sb_pack *pack = nullptr; // observations and redshifts are fixed over the fit: precompute once (fp32 fast path)
    int32_t launches = 0;
    if (base == SB_F32 && sb_pack_observations(m, b, &db, (void *)st, &pack) == SB_OK) { db.pack = pack; launches += tl_launches; }
    sb_fit_result dres;
    dres.theta = D + r_theta; dres.chi2 = D + r_chi2;
    dres.status = (int32_t *)(D + r_status); dres.n_iter = (int32_t *)(D + r_iter); dres.n_eval = (int32_t *)(D + r_eval);
    dres.trace = opts->trace_len > 0 ? (double *)(D + r_trace) : nullptr;
    rc = fit_device(m, b, &db, D + o_flux, D + o_err, opts, &dres, st);
    launches += tl_launches;
    const int32_t form = tl_form;
    d2h(hres->theta, r_theta, 4 * es * nun); d2h(hres->chi2, r_chi2, es * nun);
    d2h(hres->status, r_status, 4 * nun); d2h(hres->n_iter, r_iter, 4 * nun); d2h(hres->n_eval, r_eval, 4 * nun);
    if (opts->trace_len > 0) d2h(hres->trace, r_trace, 8 * (size_t)opts->trace_len * nun);
    if (!cuda_ok(cudaStreamSynchronize(st)) && rc == SB_OK) rc = SB_ECUDA;
    sb_free_pack(pack);
    tl_launches = rc == SB_OK ? launches : 0;
    tl_form = rc == SB_OK ? form : 0;
    return rc;
}

} // extern "C"
