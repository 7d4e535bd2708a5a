/*
 * sh.h -- C ABI of the Shack-Hartmann spot-and-centroid path (part of libpyr.so).
 *
 * The second FFT workload of arxiv/paper_2602_06688: the `SH` processing object
 * followed by `ShSlopec` (Table 4), whose cost the paper gives as
 * "n_subapertures x FFT x FFT" (Table 2).  The paper prints no formula; the
 * definition implemented is the one of oracle/sh_oracle.c:
 *
 *   n_sub x n_sub lenslets over the N_pup x N_pup pupil, p = N_pup / n_sub pixels each;
 *   f = DFT2_F(zero-pad(A exp(i phi) on the p x p patch)), sign -, unnormalised;  S = |f|^2 / F^2;
 *   c(u) = u (u < F/2) else u - F;  flux = sum S;  mx = sum c(u) S (u != F/2), my likewise;
 *   valid iff sum A^2 >= 0.5 p^2;  slopes = (mx, my) / flux in focal samples (one sample = a tilt of
 *   2 pi / F rad per pupil pixel), 0 where invalid;
 *   optional detector image: the centred spot (U = c(u) + F/2) summed over bs x bs blocks.
 *
 * Plain pointers and sizes, no torch types; device pointers unless stated.  sh_compute is
 * asynchronous on `stream`, allocates nothing, never synchronises, is CUDA-graph capturable and
 * deterministic (no atomics).  There is no CPU fallback.
 */
#ifndef SH_H
#define SH_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct sh_plan sh_plan; /* opaque */

/*
 * N_pup P : pupil side in pixels;  n_sub : lenslets across, divides P, p = P / n_sub <= 32;
 * F : focal-plane samples per sub-aperture side, any even number with max(p, 4) <= F <= 512 (the paper's 56, 68
 *     and 240, Table 2, are not powers of two); p = 4, 8 or 16 with p | F and
 *     spot_binning | F/p takes the pruned-transform kernel, everything else the direct contraction;
 * spot_binning bs >= 1, divides F (detector pixels n_pix = F / bs across a sub-aperture);
 * batch B >= 1 pupils per call.  Returns NULL on failure (sh_last_error / sh_last_error_string;
 * codes as in pyr.h: 1 bad argument, 2 unsupported, 3 out of memory, 4 CUDA error).
 */
sh_plan *sh_plan_create(int N_pup, int n_sub, int F, int spot_binning, int batch);

/*
 * amp, phase : device, const, [B][P][P] float32 (phase in radians).
 * out_slopes : device, [B][2][n_sub][n_sub], plane 0 = sx, plane 1 = sy; overwritten.
 * out_flux   : device, [B][n_sub][n_sub], or NULL.
 * out_spots  : device, [B][n_sub][n_sub][n_pix][n_pix], or NULL.
 * Returns 0, 1 (NULL plan / amp / phase / out_slopes, or the current device is not the plan's) or 4 (launch failed).
 */
int sh_compute(sh_plan *plan, const float *amp, const float *phase, float *out_slopes, float *out_flux,
               float *out_spots, void *stream);

/* NULL is a no-op.  The caller must have synchronised the stream(s) the plan was used on. */
void sh_plan_destroy(sh_plan *plan);

int sh_last_error(void);
const char *sh_last_error_string(void);

#ifdef __cplusplus
}
#endif
#endif /* SH_H */
