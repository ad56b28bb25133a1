// sb_internal.h -- private definitions of libsaltband (handles, kernel parameter blocks).
// Product code: shares nothing with oracle/.  Public ABI: include/saltband.h.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "saltband.h"

#define SB_MAX_CL 8
// Device model tables: node l of a phase row lives at column l + SB_PAD_L; the row is zero padded
// on both sides so that the kernels' aligned loads of a node window that starts on the grid stay inside
// the row without bounds checks: 8 columns on the left (windows start at node >= -4), a whole 256-node
// window plus slack on the right.  ld = round_up(n_wave + SB_PAD_L + SB_PAD_R, 4).
#define SB_PAD_L 8
#define SB_PAD_R 272

// Physical constants (CGS, Angstrom) -- PAPER.md:41 "h and c are the Planck constant and the speed
// of light"; AB reference flux density for the zero point (G7).
#define SB_H_PLANCK 6.62607015e-27
#define SB_C_ANGSTROM 2.99792458e18
#define SB_AB_FNU 3.631e-20

// Model geometry + colour law, passed to kernels by value.
struct SbModelParams {
    int32_t n_phase, n_wave, ld, n_cl; // ld = row stride (elements) of the device tables
    double p0, dp;                     // phase grid origin / step (days)
    double l0, dl;                     // wavelength grid origin / step (Angstrom, rest frame)
    double cl[SB_MAX_CL];              // colour-law coefficients, zero padded
    double cl_b, cl_inv_span;          // reduced wavelength r = (l - cl_b) * cl_inv_span
    double r_lo, r_hi;                 // images of cl_lo, cl_hi
    double p_lo, s_lo, p_hi, s_hi;     // polynomial value and slope at r_lo, r_hi
    double inv_dp;                     // 1 / dp (the tiled kernel multiplies instead of dividing)
};

// Interleaved {M0, M1} fp32 table of the band-grouped kernel (sb_hoist.cuh): [n_phase][SBH_LDN]
// float2, node l at column l + SBH_PAD_L, zero padded.  The row stride is a compile-time constant so
// that the four phase rows of a cell are reached with immediate offsets from one pointer.
#define SBH_PAD_L 16
#define SBH_LDN 1856

// fp32 tables of the node-weight kernel (sb_nw.cuh) in ONE allocation: M0 [n_phase][ld] at byte 0 and M1
// [n_phase][ld] at the compile-time byte offset SBN_M1_OFF (node l at column l + SB_PAD_L, zero padded), so
// that the M1 row of a phase is reached from the pointer to its M0 row with an immediate offset (global loads
// take signed 24-bit immediates: < 8 MB).  Models whose M0 table exceeds SBN_M1_OFF run the direct kernel.
#define SBN_M1_OFF (4 << 20)

struct sb_model {
    SbModelParams prm;
    float *m0_f32, *m1_f32;   // [n_phase][ld], zero padded (SB_PAD_L)
    double *m0_f64, *m1_f64;  // [n_phase][ld]
    float2 *m01_f32;          // [n_phase][SBH_LDN] or NULL when n_wave + 34 > SBH_LDN
    float *mx_f32;            // M0 table, M1 table SBN_M1_OFF bytes further (see above); NULL if M0 exceeds the offset
    int device;
    int n_sm, smem_optin;     // of `device`, read once at load
};

struct SbScratch;             // saltband.cu: per-stream workspaces and host-call contexts of a bands handle

struct sb_bands {
    int32_t n_bands, n_total, max_n;
    int32_t *d_off;        // [n_bands+1]
    double *d_lam_first;   // [n_bands] first wavelength of each band grid
    double *d_zpab_inv;    // [n_bands] 1 / ZPAB_b
    float2 *d_tab_f32;     // [n_total] {lam_j - lam_first, folded weight w_j T_j lam_j/(hc)}
    double2 *d_tab_f64;
    double *h_zpab;        // host copy [n_bands]
    double max_span;       // max over bands of (lam_last - lam_first)
    // band-grouped kernel (sb_hoist.cuh): only when every band grid is uniform
    int32_t all_uniform;   // 1 when |lam_j - (lam_first + j h_b)| <= 1e-9 lam_j for every band
    float *d_w_f32;        // [n_total] folded weights
    float2 *d_wd_f32;      // [n_total] {folded weight, lam_j - (lam_first + j h_b)}: node-weight kernel, non-uniform grids
    double *d_dlam_f64;    // [n_total] lam_j - lam_first
    double *d_h;           // [n_bands] mean step h_b = (lam_last - lam_first)/(n - 1) (the step, when the grid is uniform)
    int device;
    SbScratch *scratch;    // owned; the only mutable part of the handle (a cache, guarded by its mutex)
};

// Pack (sb_pack_observations): everything the node-weight kernel needs that does not depend on theta.
struct sb_pack {
    int32_t n_sn, n_bands;
    int32_t *d_perm;        // [n_sn] supernova indices in redshift order (stable counting sort)
    void *d_geom;           // [n_sn][n_bands] sbn::NItem
    unsigned char *d_ws;    // build workspace of the z-order sort (kept: the build is stream ordered)
    const sb_model *model;  // identity of the handles the pack was built from
    const sb_bands *bands;
    const void *z;          // the batch's redshift array the pack was built from (identity check only)
    int device;
};

// Kernel parameter block.
struct SbKParams {
    SbModelParams mp;
    const void *m0, *m1;              // tables of the kernel's real type
    int32_t n_bands, n_band_total;
    const int32_t *band_off;
    const double *band_lam_first, *band_zpab_inv;
    const void *band_tab;             // interleaved {dlam_j, W_j} pairs of the kernel's real type
    int32_t n_sn, n_samples;
    const int32_t *obs_offset;
    const void *time, *zp, *z, *x0, *x1, *c, *t0;
    const int32_t *band;
    const void *flux, *fluxerr;       // may be NULL
    void *out_flux, *out_dflux, *out_chi2, *out_dchi2; // may be NULL
    int32_t tile_cells;               // coefficient-row entries per warp buffer (multiple of 8)
    int32_t chunk_cap;                // evaluation records per chunk
    int32_t group_units;              // units per CTA group (<= 16)
    const int32_t *n_live;            // fit driver: [1] 0 = nothing to do (or NULL)
};

// Kernel parameter block of the band-grouped kernel (sb_hoist.cuh), fp32 forward.
struct SbHParams {
    SbModelParams mp;
    const float2 *m01;                // [n_phase][SBH_LDN] {M0, M1}
    const float *m0, *m1;             // [n_phase][mp.ld] (unused by the grouped kernel; kept for layout)
    int32_t n_bands, n_band_total;
    const int32_t *band_off;
    const double *band_lam_first, *band_zpab_inv, *band_h, *band_dlam;
    const float *band_w;
    int32_t n_sn, n_samples;
    const int32_t *obs_offset;
    const float *time, *zp, *z, *x0, *x1, *c, *t0;
    const int32_t *band;
    const float *flux, *fluxerr;      // may be NULL
    float *out_flux, *out_chi2;       // may be NULL
    float *out_dflux, *out_dchi2;     // gradient kernel only; may be NULL
    const int32_t *perm;              // z-ordered supernova indices (workspace) or NULL
    unsigned int *counter;            // group counter (workspace, zeroed by sb_zorder_kernel)
    int32_t group_units;              // units per group (<= 32)
    int32_t cap;                      // observations per round
};
