/*
 * chain.h -- C ABI of the steps either side of the wavefront sensor (part of libpyr.so):
 * the on-device phase source, the detector model, the pupil-map calibrator, slopes from detector pixels and
 * the modal reconstructor, so that in a loop step only the reconstructed modes leave the device.
 *
 * arxiv/paper_2602_06688 names these processing objects and their parameters and prints no formula for any of
 * them (Table 4, PAPER.md:311-315 `AtmoEvolution` / `AtmoPropagation`, 323 `CCD`, 327 `PyrSlopec`, 332 `Modalrec`,
 * 337 `PyrPupdataCalibrator`; Listing 2, PAPER.md:476-514 atmosphere and propagation blocks, 557-589 detector
 * block, 592-604 slope computer, 606-612 reconstructor).  The definitions implemented are those of
 * oracle/chain_oracle.c (readings A1-A4, C1-C7, U1, M1).
 *
 * Plain pointers and sizes, no torch types; "device" = device memory of the CUDA device that was current when
 * the plan was created, "host" = host memory.  Every *_compute / atmo_propagate / ccd_integrate call is
 * asynchronous on `stream`, allocates nothing, never synchronises, is CUDA-graph capturable and deterministic
 * (no atomics).  There is no CPU fallback.  Error codes as in pyr.h (0 ok, 1 bad argument, 2 unsupported,
 * 3 out of memory, 4 CUDA error); chain_last_error / chain_last_error_string describe the last failure of the
 * calling thread.
 */
#ifndef CHAIN_H
#define CHAIN_H

#ifdef __cplusplus
extern "C" {
#endif

/* ---------------------------------------------------------------- AtmoEvolution + AtmoPropagation
 * phase[b][y][x] = sum_l w_l bilerp(screen_l, y + dy[b][l], x + dx[b][l]),  0 <= y, x < N_pup:
 * n_layers periodic S x S phase screens (radians at the sensing wavelength, pupil pixel pitch), each displaced
 * by a real number of pixels (wind speed x time / pitch + layer height x source direction / pitch; the caller
 * computes it) and interpolated bilinearly with periodic wrap; geometric propagation = sum. */
typedef struct atmo_plan atmo_plan;

/* n_layers >= 1, screen_side S >= 2, N_pup >= 1, batch B >= 1 sources, n_layers * batch <= 128.  NULL on failure. */
atmo_plan *atmo_plan_create(int n_layers, int screen_side, int N_pup, int batch);
/* host_weights: [n_layers] or NULL (all 1). */
int atmo_plan_set_weights(atmo_plan *plan, const float *host_weights);
/* screens: device, const, [n_layers][S][S] float32.  host_shift_yx: HOST, [B][n_layers][2] doubles (dy, dx) in
 * pixels, read before the call returns (split into floor and fraction in double; captured by value in a graph).
 * out_phase: device, [B][N_pup][N_pup] float32, overwritten. */
int atmo_propagate(atmo_plan *plan, const float *screens, const double *host_shift_yx, float *out_phase, void *stream);
void atmo_plan_destroy(atmo_plan *plan);

/* ---------------------------------------------------------------- CCD
 * One call = one simulation step: acc += flux_gain * intensity (expected photo-electrons; float32 fma).  Every
 * n_int-th call reads the frame out and clears acc: photon noise (Poisson: inversion below 30 e-, rounded normal
 * approximation above), readout noise (normal, sigma = readout_level e-), ADC (adu_gain > 0: divide by adu_gain
 * [e-/ADU], round to nearest, clamp to [0, 2^n_bits - 1]; adu_gain = 0: electrons as float).  Random numbers:
 * Philox4x32-10, counter (pixel index, frame index, 0, 0), key = seed -- reproducible bit for bit
 * (`dt`, `photon_noise`, `readout_noise`, `readout_level`, `quantum_eff`). */
typedef struct ccd_plan ccd_plan;

/* n_pixels: pixels per call over all sources (B * N_det * N_det), 1 <= n_pixels < 2^32; n_int >= 1;
 * readout_level >= 0; adu_gain >= 0; 1 <= n_bits <= 30.  NULL on failure. */
ccd_plan *ccd_plan_create(long long n_pixels, int n_int, int photon_noise, int readout_noise, float readout_level,
                          float adu_gain, int n_bits, unsigned long long seed);
/* intensity: device, const, [n_pixels] float32.  out_pixels: device, [n_pixels] float32, written only when a frame
 * is read out.  *frame_ready (host, may be NULL) = 1 if this call read a frame out, else 0 (known on the host:
 * the step counter lives in the plan). */
int ccd_integrate(ccd_plan *plan, const float *intensity, float flux_gain, float *out_pixels, int *frame_ready, void *stream);
/* Restart: clears the accumulator (asynchronously on `stream`) and the step / frame counters. */
int ccd_reset(ccd_plan *plan, void *stream);
void ccd_plan_destroy(ccd_plan *plan);

/* test-only: raw generator output for counters (i, frame, 0, 0), i < n: device out_words [n][4] uint32 */
int ccd_test_philox(unsigned long long seed, unsigned int frame, long long n, unsigned int *out_words, void *stream);

/* ---------------------------------------------------------------- PyrPupdataCalibrator
 * valid[Y][X] = [ T[Y][X] >= threshold * max T ],  T = (Qa + Qb) + (Qc + Qd) of a reference detector frame
 * (float32), N_det even, N_q = N_det / 2 (tag `th0.30` at PAPER.md:596).  Calibration-time call:
 * synchronises `stream`.  ref_frame: device [N_det][N_det]; host_valid_out: HOST [N_q][N_q] bytes, for
 * pyr_plan_set_valid / modalrec_plan_create. */
int pupdata_from_frame(int N_det, const float *ref_frame, float threshold, unsigned char *host_valid_out, void *stream);

/* ---------------------------------------------------------------- Modalrec
 * modes[b][m] = sum_i R[m][i] sv[b][i],  sv = [sx at the valid pixels in row-major (Y, X) order, then sy likewise]
 * (PAPER.md:332, 606-612).  float32 storage, float32 FMA accumulation in a fixed order. */
typedef struct modalrec_plan modalrec_plan;

/* host_valid: HOST [N_q][N_q] bytes; host_recmat: HOST [n_modes][2 n_valid] float32 (copied).  batch B >= 1.
 * Up to about 50 000 slopes (2 n_valid): beyond 8192 the slope vectors of the sources that share one pass over R sit in
 * shared memory (four sources per pass if they fit, else fewer); more slopes than fit give error 2. */
modalrec_plan *modalrec_plan_create(int n_modes, int N_q, const unsigned char *host_valid, const float *host_recmat, int batch);
/* slopes: device, const, dense [B][2][N_q][N_q] float32 (the layout pyr_compute writes).  out_modes: device [B][n_modes]. */
int modalrec_compute(modalrec_plan *plan, const float *slopes, float *out_modes, void *stream);
void modalrec_plan_destroy(modalrec_plan *plan);

int chain_last_error(void);
const char *chain_last_error_string(void);

#ifdef __cplusplus
}
#endif
#endif /* CHAIN_H */
