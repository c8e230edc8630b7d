/* tomo_host.h -- host-only entry points of libtomo_b200 (no CUDA device needed).
 *
 * They expose row A0 of DESIGN.md -- the one-time covariance-kernel builder -- so that it can be checked on a CPU
 * box against an independent evaluation of the same paper formulas (
 * Eq.50-53).  All pointers are HOST pointers; outputs are caller-allocated fp64 arrays.  Return codes and
 * tomo_last_error() as in tomo.h.
 */
#ifndef TOMO_B200_HOST_H
#define TOMO_B200_HOST_H
#include "tomo.h"
#ifdef __cplusplus
extern "C" {
#endif

/* Sizes the plan would use: valid subapertures / phase points (Fig.2, reading G12), n' (L179, G19),
 * FFT edges P, P_os (L207, G11) and the number of layer tables kept apart in the phi-s product (K or 1). */
int tomo_host_sizes(const tomo_geometry *geom, const tomo_cn2 *cn2, int pad, int pad_os, int *n_vs, int *n_vphi,
                    int *n_prime, int *P, int *P_os, int *Kp);

/* theta[(i,a),(j,b)](l): gen_out[C][C][2n-1][2n-1], index (ly+n-1, lx+n-1), lag = input - output (L150, L265). */
int tomo_host_css_generators(const tomo_geometry *geom, const tomo_cn2 *cn2, double r0, double L0, int slope_model,
                             double *gen_out);

/* xi'[k,(j,b)](l) of one target: gen_out[Kp][C][n'+n-1][n'+n-1], l = q - p' (L193-197, reading G18). */
int tomo_host_cos_generators(const tomo_geometry *geom, const tomo_cn2 *cn2, double r0, double L0, int slope_model,
                             int target, double *gen_out);

/* Generators of a layered plan (tomo_options.layered, L199; reading G31): xi'[k,(j,b)](l) on the n_m x n_m grid of every
 * layer, centred on the axis: gen_out[K][C][n_m+n-1][n_m+n-1], l = q - m.  *n_m_out receives n_m for fov_radius [arcsec];
 * gen_out may be NULL to query n_m alone.  geom->n_targets must be 0. */
int tomo_host_layer_generators(const tomo_geometry *geom, const tomo_cn2 *cn2, double r0, double L0, int slope_model,
                               double fov_radius, int *n_m_out, double *gen_out);

/* Spectrum of one generator gen[n_out+n_in-1][n_out+n_in-1]: circular embedding at edge P, 2-D real DFT, times
 * 1/P^2, Hermitian half: spec_out[P/2+1 (kx)][P (ky)][2 (re, im)]  (L207, L265; readings G10, G24). */
int tomo_host_generator_spectrum(const double *gen, int n_out, int n_in, int P, double *spec_out);

/* D_phi(r) of Eq.53 (L619) for count separations r [m]. */
int tomo_host_structure_function(const double *r, int count, double r0, double L0, double *out);

/* Low-order NGS tip/tilt estimator of tomo_lo_create (reading G30; L321, L412) without a device.  M = n_lo + n_targets
 * directions, sensors first.  R_out: host [2 n_targets][2 n_lo] row-major, order [direction][x, y]; cov_out: host [2M][2M]
 * covariance of the aperture-mean slope pairs (without the noise term).  Either may be NULL. */
int tomo_host_lo_estimator(const tomo_geometry *geom, const tomo_cn2 *cn2, double r0, double L0, int slope_model,
                           double sigma2_lo, double *R_out, double *cov_out);

/* Work table of the persistent solver's batch path: how the Ph x n_frames slab passes of one CG iteration (one k_x slab of
 * all channels of one frame: y-FFTs + the per-frequency block product, Eq.22 / Eq.30) are dealt to n_ctas CTAs.  CTA b
 * owns slab b % Ph with the other CTAs of that residue; CTAs above the average hand frames to CTAs below it (one helped
 * slab per CTA).  seg_out: host int [n_ctas][8] = {own f_lo, own f_hi, helped k_x, helped f_lo, helped f_hi, 0, 0, 0}. */
int tomo_host_slab_segments(int Ph, int n_frames, int n_ctas, int *seg_out);

#ifdef __cplusplus
}
#endif
#endif
