/*
 * pyr.h -- C ABI of libpyr: modulated pyramid wavefront-sensor propagation on one B200.
 *
 * The operation is the hot path named by BASELINE.json:north_star: what SPECULA's
 * `ModulatedPyramid` processing object computes in its `trigger`, followed by the
 * arithmetic of `PyrSlopec` (paper: Table 4; parameters in
 * Listing 2; FFT workload `n_mod x N_fft x N_fft`,
 * Table 2).  The paper prints no formula for the sensor; the exact
 * definition implemented is SURVEY.md section 8(c) steps 1-10 (restated in DESIGN.md):
 *
 *   for every source s and modulation point k = 0..n_mod-1 (theta_k = 2 pi k / n_mod):
 *     E_k = amp * exp(i (phase + tilt_k)),   zero-padded, centred, to N_fft x N_fft
 *     F_k = DFT2(E_k)                         (sign -, unnormalised)
 *     O_k = IDFT2(F_k * mask) / N_fft^2       (four-face pyramid mask (-i)^(|fu|+|fv|))
 *   I = sum_k |O_k|^2 ;  D = binning x binning block sums of I ;
 *   slopes: sx = ((Qb+Qd)-(Qa+Qc))/T,  sy = ((Qc+Qd)-(Qa+Qb))/T on valid pixels, 0 elsewhere,
 *   with Qa,Qb,Qc,Qd the (low y,low x), (low y,high x), (high y,low x), (high y,high x)
 *   quadrants of D and T the mean of Qa+Qb+Qc+Qd over the valid pixels.
 *
 * Execution rules follow the paper's `trigger` contract: pyr_compute
 * allocates nothing, never synchronises, and may be captured in a CUDA graph.
 *
 * All arrays are dense, row-major [y][x] with x fastest, float32.  "device" pointers are
 * CUDA device memory of the device that was current at pyr_plan_create; "host" pointers
 * are ordinary (preferably pinned) host memory.  The caller owns every data pointer; the
 * library never frees or retains them beyond the enqueued work.  The plan owns its tables
 * and workspace.  One plan may be used from one stream at a time.
 *
 * Every function is thread-safe with respect to other plans.  No C++ exception crosses the
 * boundary.  There is no CPU fallback: without a CUDA device pyr_plan_create fails with
 * PYR_ECUDA.
 */
#ifndef PYR_H
#define PYR_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct pyr_plan pyr_plan; /* opaque */

enum {
    PYR_OK = 0,
    PYR_EINVAL = 1,       /* bad argument */
    PYR_EUNSUPPORTED = 2, /* valid request the kernels do not cover */
    PYR_ENOMEM = 3,       /* host or device allocation failed */
    PYR_ECUDA = 4         /* CUDA runtime error (no device, launch failure, ...) */
};

/*
 * Create a plan (north_star: "a plan holding precomputed twiddle tables, tilt phasors and
 * the pyramid mask").  Tables are computed in double on the host and rounded once to
 * float32; all device memory the plan will ever need is allocated here.
 *
 *   N_pup    P : pupil side in pixels; even, 2 <= P <= N_fft/2.  One lambda/D of tilt is
 *                2 pi of phase across P pixels (reading S10).
 *   N_fft    N : padded side; a multiple of 4, 16 <= N <= 2048.  Powers of two run the fast
 *                half-band kernels; any other N (the paper's 660 and 1600) is
 *                computed exactly by embedding the length-N circulant line operator in a cyclic
 *                convolution of the next power of two >= N + P - 1, which must be <= 2048
 *                (else PYR_EUNSUPPORTED).
 *   n_mod    M : number of modulation points, >= 1, equally spaced on a circle, theta_0 = 0,
 *                weight 1 each (reading S9).
 *   r_mod_lambda_over_D : circle radius in lambda/D, finite, >= 0.
 *   binning  b : detector binning; b >= 1, b divides N/4 and N/4 - P/2 (pupil images
 *                align with the detector grid).  N_det = N/b, N_q = N_det/2.
 *   batch    B : sources per pyr_compute call, >= 1.
 *
 * Returns NULL on failure; pyr_last_error() / pyr_last_error_string() tell why
 * (PYR_EINVAL for the constraints above, PYR_ENOMEM, PYR_ECUDA).
 */
pyr_plan *pyr_plan_create(int N_pup, int N_fft, int n_mod, float r_mod_lambda_over_D,
                          int binning, int batch);

/*
 * As pyr_plan_create, for an arbitrary set of modulation points instead of the circle: point k
 * adds weight[k] * |O_k|^2 with the tilt (ax[k], ay[k]) in lambda/D (x, y; one lambda/D = 2 pi of
 * phase across N_pup pixels, reading S10) -- extended or off-axis sources, non-circular modulation
 * paths (the `ExtendedSource` and modulated sensors of Table 4).
 * ax, ay: host, [n_points] float32, finite; weight: host, [n_points] float32 >= 0, or NULL for 1.
 * Points with exactly equal ay share one y-pass.  pyr_plan_create(P, N, M, r, b, B) is the special
 * case ax = r cos(2 pi k / M), ay = r sin(2 pi k / M), weight 1.  Same errors as pyr_plan_create.
 */
pyr_plan *pyr_plan_create_points(int N_pup, int N_fft, int n_points, const float *ax, const float *ay,
                                 const float *weight, int binning, int batch);

/*
 * PolyCromPyramid (Table 4; reading PC1): the sensor
 * sums the intensities of n_wavelengths wavelengths.  amp and phase are given at the reference wavelength
 * lambda_0; at wavelength l the optical path is the same, so the whole pupil phase -- turbulence and modulation
 * tilt -- is scaled by ratio[l] = lambda_0 / lambda_l while the sampling (N_pup, N_fft) and the mask stay:
 *   I = sum_l weight[l] sum_k | IDFT2( mask . DFT2( A exp(i ratio[l] (phi + tilt_k)) ) ) |^2,
 * k over the modulation circle (n_mod, r_mod in lambda_0 / D).  ratio: host, [n_wavelengths] float32, finite,
 * > 0, pairwise different; weight: host, [n_wavelengths] float32 >= 0, or NULL for 1.  The wavelength is one more
 * accumulation axis of the same kernels (n_mod * n_wavelengths tasks per row).  Same errors as pyr_plan_create.
 */
pyr_plan *pyr_plan_create_poly(int N_pup, int N_fft, int n_mod, float r_mod_lambda_over_D, int n_wavelengths,
                               const float *ratio, const float *weight, int binning, int batch);

/*
 * ModulatedDoubleRoof (Table 4; reading DR1): two roof
 * prisms in two focal planes instead of the four-face pyramid -- roof 1 splits along x, mask1[v][u] = (-i)^|f(u)|;
 * the propagation from its focal plane to the second one is the pupil-plane factor
 * q[y][x] = exp(i pi kappa ((x - c)^2 + (y - c)^2)), c = (N_fft - 1)/2 (kappa in 1/pixel^2); roof 2 splits along y.
 * enable != 0 switches the plan to this sensor, enable == 0 back to the pyramid (kappa = 0 IS the pyramid).
 * The slopes are those of the four pupil images as before (`DoubleRoofSlopec`).  Host call (re-uploads two small
 * tables); not for polychromatic plans (PYR_EUNSUPPORTED) nor while a custom mask is set (PYR_EINVAL).
 */
int pyr_plan_set_double_roof(pyr_plan *plan, int enable, float kappa);

/*
 * Launch schedule of the ELT-scale size (N_fft = 2048; north_star item (3) "the working set stays L2-resident").
 * l2_resident = 0 (default): one column-pass launch over all y-tilts, one row-pass launch; the intermediate R
 * (0.38 GB at C5) goes through HBM once each way.  l2_resident != 0: the two passes run per chunk of j_per_chunk
 * y-tilts (<= 0: chosen so that two chunks of R fit 80 MB); R is a ring of two chunks that is overwritten while still
 * in L2, the row pass leaves one partial frame per chunk in S and k_rebin sums them.  Same results up to the
 * float32 summation order over chunks; 2 x chunks + 2 launches per call.  Measured slower at C5;
 * kept as an option and as the evidence.  PYR_EUNSUPPORTED for other sizes.  Host call; may allocate (S slots).
 */
int pyr_plan_set_schedule(pyr_plan *plan, int l2_resident, int j_per_chunk);

/*
 * Enqueue one pass of the whole path on `stream` (a cudaStream_t; NULL = legacy default
 * stream) and return without waiting.
 *
 *   amp           device, const, [batch][N_pup][N_pup]; >= 0, finite.  The library applies no
 *                 pupil stop of its own: zero amplitude outside the pupil is the caller's job.
 *   phase         device, const, same shape, radians at the sensing wavelength (reading S12);
 *                 must be finite everywhere (values where amp == 0 do not matter).
 *   out_intensity device, [batch][N_det][N_det]; overwritten with D.  May be NULL.
 *   out_slopes    device, [batch][2][N_q][N_q], plane 0 = sx, plane 1 = sy; overwritten.
 *                 May be NULL.  At least one output must be non-NULL.
 *
 * Returns PYR_OK, PYR_EINVAL (NULL plan/amp/phase, both outputs NULL) or PYR_ECUDA (a launch
 * failed; the message holds cudaGetErrorString).  Results are deterministic: the same inputs
 * give bit-identical outputs on every call (no atomics on the data path).
 */
int pyr_compute(pyr_plan *plan, const float *amp, const float *phase, float *out_intensity,
                float *out_slopes, void *stream);

/*
 * PyrSlopec on detector pixels (the slope computer takes `detector.out_pixels`): steps
 * 8-10 of the definition applied to a detector frame instead of the noise-free intensity -- quadrants, the plan's
 * validity map (pyr_plan_set_valid; a threshold-derived one comes from pupdata_from_frame, chain.h), global-mean
 * normalised slopes.  pixels: device, const, [B][N_det][N_det] float32 (e.g. the output of ccd_integrate);
 * out_slopes: device, [B][2][N_q][N_q], overwritten.  Asynchronous on `stream`, no allocation, no synchronisation.
 */
int pyr_slopes_from_pixels(pyr_plan *plan, const float *pixels, float *out_slopes, void *stream);

/*
 * The same operation (steps 8-10 on a detector frame) for callers that cannot allocate device
 * memory and so cannot create a plan: code under CUDA graph capture, tight serving loops, harnesses that forbid
 * cudaMalloc.  No plan; this call allocates nothing (no cudaMalloc, cudaFree or allocating library routine): its
 * scratch, the [batch][N_det] row sums over valid pixels, lives in a static device array of 65536 floats (256 KB)
 * that every GPU loading the library holds until the process exits.
 *   N_det   detector side, even, >= 2; N_q = N_det / 2.  batch: 1..65535 frames.
 *   LIMIT   batch * N_det <= 65536, else PYR_EUNSUPPORTED (use a plan and pyr_slopes_from_pixels).
 *   pixels  device, const, [batch][N_det][N_det] float32.
 *   valid   device, const, [N_q][N_q] bytes (non-zero = valid); n_valid: the number of non-zero entries (the caller
 *           counts them once; 0 gives all-zero slopes, as in the plan path).
 *   out_slopes  device, [batch][2][N_q][N_q] float32, overwritten.
 * Asynchronous on `stream`, never synchronises; results are bit-identical to pyr_slopes_from_pixels with the same
 * validity map.  ALL calls in the process (on one device) share the one scratch array: calls that may overlap on the
 * GPU -- different streams without an ordering between them -- race on it; keep them on one stream or order them with
 * events.  The array keeps the last call's row sums; every entry a call reads it has written first, so nothing needs
 * clearing.  pyr_static_scratch_init() resolves the array's device address for the current device (done by the first
 * call otherwise; call it once per device before a graph capture).  PYR_ECUDA if the address cannot be resolved.
 */
int pyr_slopes_from_pixels_static(int N_det, int batch, const float *pixels, const unsigned char *valid, int n_valid,
                                  float *out_slopes, void *stream);
int pyr_static_scratch_init(void);

/*
 * End-to-end variant with HOST buffers (same shapes and meaning as pyr_compute): copies
 * amp/phase host->device, runs the path, copies the requested outputs device->host, and
 * returns after the stream has completed.  Uses staging buffers owned by the plan.
 */
int pyr_compute_host(pyr_plan *plan, const float *amp_host, const float *phase_host,
                     float *out_intensity_host, float *out_slopes_host, void *stream);

/*
 * Double-buffered end-to-end variant for a loop that feeds host inputs every step: enqueue and return.  slot = 0 or
 * 1 selects one of two staging sets owned by the plan; the H2D copy of amp / phase, the kernels and the D2H copy of
 * the requested outputs run on three internal streams chained by events, so the copies of call i + 1 overlap the
 * kernels of call i (calls execute in the order they were enqueued; the kernels of different calls never overlap).
 * The host buffers must be pinned for the copies to be asynchronous, must stay valid and -- the outputs --
 * untouched until pyr_host_wait(plan, slot) has returned, and a slot must be waited for before it is enqueued again.
 * pyr_host_wait blocks until the outputs of the last call on `slot` are in host memory (PYR_OK at once if none).
 * Not to be mixed with pyr_compute / pyr_compute_host on the same plan while calls are in flight.
 */
int pyr_compute_host_async(pyr_plan *plan, const float *amp_host, const float *phase_host, float *out_intensity_host,
                           float *out_slopes_host, int slot);
int pyr_host_wait(pyr_plan *plan, int slot);

/* Destroy a plan.  NULL is a no-op.  The caller must have synchronised the stream(s) the plan
 * was used on. */
void pyr_plan_destroy(pyr_plan *plan);

/*
 * Replace the sub-aperture validity map (default: pixel centre inside the geometric
 * pupil-image circle).  host_valid: host, [N_q][N_q] bytes, non-zero =
 * valid.  Synchronous (blocks until the table is on the device).  PYR_EINVAL on NULL.
 */
int pyr_plan_set_valid(pyr_plan *plan, const unsigned char *host_valid);

/*
 * Replace the focal-plane mask by a separable one, mask[v][u] = gy[v] * gx[u].  gx, gy: host,
 * [N_fft][2] float32 (re, im), natural DFT frequency order.  The default pyramid is the
 * separable mask gx[u] = gy[u] = (-i)^|f(u)|.  Used by the identity-mask and pure-shift-mask
 * parity tests (pins P4, P5); selects the table-driven (slower) mask multiply.  Passing
 * NULL for both restores the built-in pyramid.  Synchronous.
 */
int pyr_plan_set_mask_separable(pyr_plan *plan, const float *gx_ri, const float *gy_ri);

/*
 * Replace the focal-plane mask by an arbitrary complex N_fft x N_fft one (field stop, face or
 * edge defects, other pupil separations: the generalisations SURVEY.md 8(f) lists for the
 * ModulatedPyramid family).  mask_ri: host, [N_fft][N_fft][2] float32
 * (re, im), mask[v][u] in natural DFT frequency order (v = y frequency, u = x frequency), the
 * factor applied to the un-normalised forward DFT before the inverse DFT (SURVEY.md 8(c) steps
 * 3-5).  Selects the general three-pass path (forward x | forward y, mask, inverse y | inverse
 * x), which processes the modulation points in chunks; on first use it allocates its
 * workspace (a device copy of the mask and two spectra buffers of at most ~0.7 GB), so call it
 * outside any timed region or graph capture.  NULL restores the mask that was active before
 * (built-in pyramid or separable).  Synchronous.  PYR_EINVAL, PYR_ENOMEM, PYR_ECUDA.
 */
int pyr_plan_set_mask(pyr_plan *plan, const float *mask_ri);

/* Query derived sizes; any output pointer may be NULL. */
int pyr_plan_get_dims(const pyr_plan *plan, int *N_det, int *N_q, int *n_valid);

/*
 * Test-only export (not on the timed path): apply the 1-D operator
 *   out = IDFT_N( g * DFT_N( zero-pad(in, N) ) ) / N
 * to `nlines` independent lines with the plan's x-mask, through the same device routine the
 * row pass uses.  in: device, [nlines][N_pup][2] float32; out: device, [nlines][N_fft][2].
 */
int pyr_test_line_conv(pyr_plan *plan, const float *in_ri, float *out_ri, int nlines, void *stream);

/* How many kernels one pyr_compute call launches (for bench.py's gpu_launches). */
int pyr_plan_launches_per_compute(const pyr_plan *plan);

/*
 * Measurement hooks (bench.py only; off by default).  With profiling enabled pyr_compute records
 * a CUDA event on `stream` before and after every kernel it launches (events are created here,
 * once; recording allocates nothing and does not synchronise).  Do not capture a profiled call
 * in a CUDA graph.
 *   pyr_plan_last_kernel_ms: waits for the last profiled call to finish, writes the device
 *   time in milliseconds of its first min(n, count) kernels to ms[] (host) and returns the
 *   number of kernels that call launched, or -1 on error.
 *   pyr_kernel_name(i): name of the i-th kernel of the path ("" if out of range); static storage.
 */
int pyr_plan_set_profiling(pyr_plan *plan, int enable);
int pyr_plan_last_kernel_ms(pyr_plan *plan, float *ms, int n);
const char *pyr_kernel_name(int i);

/*
 * Measurement hook: FP32 FMA-chain microbenchmark -- 8 independent packed fma.rn.f32x2 chains per
 * thread on every SM, best of four timed launches after warm-up.  *tflops = measured FP32 throughput;
 * *sm_mhz_effective (may be NULL) = the clock at which 148 SMs x 128 lanes x 2 flop would give that number.
 * Synchronises the device; allocates and frees a scratch buffer.  bench.py prints it as roofline.peak_measured.
 */
int pyr_measure_fp32_peak(float *tflops, float *sm_mhz_effective);

/* Thread-local status of the last failing call in this thread. */
int pyr_last_error(void);
const char *pyr_last_error_string(void);

#ifdef __cplusplus
}
#endif
#endif /* PYR_H */
