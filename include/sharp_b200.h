/*
 * sharp_b200.h -- C ABI of the B200-native ptychographic projection loop of arXiv 1602.01448 (SHARP).
 *
 * The library runs steps 4-7 of the paper's "typical reconstruction" on ONE GPU:
 *   split Q, the unitary 2-D DFT F (Eq. 2), the Fourier-magnitude projection
 *   P_a (Eq. 7), the overlap Q* / Q*Q (Eq. 8-9), the RAAR frame update
 *   (step 5), the optional illumination refinement (Eq. 10) and the
 *   residuals eps_a, eps_Q, eps_Delta (Eq. 11-13).
 * Readings of the paper where it is silent or garbled are listed in DESIGN.md ("Readings", G1..G25).
 *
 * Conventions (all calls)
 *   - Arrays are row-major, C-contiguous.  Complex values are interleaved (re, im) float32 ("c64").
 *   - "dev" pointers are CUDA device pointers owned by the caller (e.g. torch tensors), on the device that owns the
 *     bound workspace and 16-BYTE ALIGNED (the kernels use 128-bit accesses; a misaligned pointer is SHARP_EINVAL);
 *     "host" pointers are ordinary host memory.  Calls may be made with any CUDA device current: the library switches
 *     to the plan's device for the duration of the call.  Inputs are consumed during the call's stream work; outputs are written into the
 *     caller's buffers.  The library never frees caller memory.
 *   - Every call returns 0 (SHARP_OK) or a negative error code; no exception or abort crosses the ABI and a
 *     call that returns SHARP_EINVAL has changed nothing.  sharp_last_error() gives the text.
 *   - Work is enqueued on the stream given to sharp_bind(); only sharp_errors(), sharp_sync() and the host-side
 *     getters synchronise.  One plan = one stream; calls on one plan are not thread-safe.
 *   - DFT convention: forward kernel exp(-2 pi i (u r + v c)/m), scale 1/m per 2-D transform each way
 *     (unitary; sign: reading G2); DC at index [0,0], no fftshift anywhere.
 *   - Positions x_i are the (row, col) of the frame's top-left pixel in the object, T_i psi(r) = psi(r + x_i)
 *     (PAPER.md:53, 68); 0 <= x_i <= obj - m on both axes, anything else is SHARP_EINVAL (no wrap-around, except in a
 *     plan made by sharp_plan_periodic).
 */
#ifndef SHARP_B200_H
#define SHARP_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define SHARP_OK 0
#define SHARP_EINVAL (-1) /* bad size, position out of range, beta outside (0.5, 1], null pointer */
#define SHARP_ESTATE (-2) /* call made before its prerequisites (bind / intensities / probe) */
#define SHARP_ENOMEM (-3) /* workspace too small, or host allocation failed */
#define SHARP_ECUDA (-4)  /* CUDA launch or runtime failure; text in sharp_last_error() */

typedef struct sharp_plan_s sharp_plan_t;

/* Edge (pixels) of the square object tiles of the gather-form overlap ("the image is divided
 * into blocks; each block determines which frames contribute"). */
#define SHARP_TILE 32

/* ---- plan -------------------------------------------------------------------------------------------------
 * sharp_plan: validates the geometry and builds the integer artefacts of step 4 on the
 * host: the copy of the positions, the per-tile CSR lists of covering frames (tiles row-major, frames in
 * ascending index), and the workspace layout.
 *   out        receives the plan (library-owned; release with sharp_destroy)
 *   m          frame edge, one of 64, 128, 256, 512
 *   K          number of frames, >= 1
 *   pos_rc     HOST, K x 2 int32, (row, col) of each frame's top-left object pixel; copied
 *   obj_rows, obj_cols   object dimensions n_r x n_c, each >= m
 * No device work is done. */
int sharp_plan(sharp_plan_t **out, int m, int K, const int32_t *pos_rc, int obj_rows, int obj_cols);
/* sharp_plan_periodic: the same with the periodic boundary of the paper's Fig. 3 simulation ("periodic
 * boundary conditions to avoid edge effects"; reading G25): T_i psi(r) = psi((r + x_i) mod n) on both axes, positions
 * anywhere in 0 <= x_i < obj, and every frame-pixel <-> object-pixel map of the library (split, overlap, tile lists,
 * cover counts, Eq. 10, residuals) wraps accordingly.  Requires obj - m >= SHARP_TILE - 1 on both axes (so that no
 * object tile meets both ends of one frame); otherwise SHARP_EINVAL.  Everything else is as for sharp_plan. */
int sharp_plan_periodic(sharp_plan_t **out, int m, int K, const int32_t *pos_rc, int obj_rows, int obj_cols);
void sharp_destroy(sharp_plan_t *p);
/* Text of the last error on this plan (or of the last failed sharp_plan if p == NULL). Never NULL. */
const char *sharp_last_error(const sharp_plan_t *p);

/* Bytes of device workspace the plan needs (frames x2, amplitudes, object-sized arrays, lists, FFT scratch). */
size_t sharp_workspace_bytes(const sharp_plan_t *p);
/* Hands the plan its device workspace (256-byte aligned, >= sharp_workspace_bytes) and the CUDA stream
 * (a cudaStream_t cast to void*; NULL = the legacy default stream).  Uploads positions and tile lists.
 * The caller keeps ownership and must keep the memory alive until sharp_destroy. */
int sharp_bind(sharp_plan_t *p, void *dev_workspace, size_t bytes, void *cuda_stream);

/* ---- inputs -----------------------------------------------------------------------------------------------
 * sharp_set_intensities: I_dev is DEVICE, K*m*m float32, frame-major, DC at [0,0] of each frame.  Stores
 * a = sqrt(max(I,0)) (clamp: reading G14) and computes ||a||^2 = sum I and the small-modulus
 * threshold thr = 1e-4 * a_rms of reading G4.  The caller may free I_dev after the stream work completes. */
int sharp_set_intensities(sharp_plan_t *p, const float *I_dev);
/* sharp_set_probe: w_dev is DEVICE, m*m c64.  Copies w and rebuilds Q*Q(p) = sum_i |w(p - x_i)|^2
 * (PAPER.md:173 step 4).  If frames already exist they are kept (they are the primary state, reading G10) and
 * the object estimate is re-evaluated under the new w. */
int sharp_set_probe(sharp_plan_t *p, const float *w_dev);
/* sharp_set_object: psi_dev is DEVICE, obj_rows*obj_cols c64, or NULL for the flat object 1+0i (reading G8).
 * Forms z^0 = Q psi^0 and resets the iteration counter.  Called implicitly with NULL by the
 * first sharp_iterate if neither it nor sharp_set_frames was called.  Needs the probe. */
int sharp_set_object(sharp_plan_t *p, const float *psi_dev);
/* sharp_set_frames: z_dev is DEVICE, K*m*m c64.  Overwrites the frame state (restore / teacher forcing);
 * the "previous iterate" of eps_Delta becomes 0 as before the first iteration. Needs the probe. */
int sharp_set_frames(sharp_plan_t *p, const float *z_dev);
/* sharp_set_frame_slots: caps the number of frames the fused per-frame kernel keeps in flight (persistent CTAs at
 * m <= 128, CTA clusters above); 0 = one per resident slot of the bound device (the default).  A tuning and test
 * hook: with fewer slots than frames every CTA loops over several frames. May be called before or after sharp_bind. */
int sharp_set_frame_slots(sharp_plan_t *p, int slots);
/* Illumination refinement every `every` iterations (Eq. 10; PAPER.md:181 "if desired", :228); 0 = fixed probe. */
int sharp_set_probe_refine(sharp_plan_t *p, int every);

/* ---- the loop ---------------------------------------------------------------------------------------------
 * sharp_iterate: n >= 0 RAAR iterations (step 5, sign of reading G1)
 *      z <- 2 beta P_Q P_a z + (1 - 2 beta) P_a z + beta (z - P_Q z),     beta in (0.5, 1]  (G15)
 * each followed by the image update psi = Q*z / Q*Q (Eq. 9, step 6) and, on iterations whose 1-based count is
 * a multiple of the refine period, the illumination update of Eq. 10 (step 7, order: reading G10).
 * Asynchronous on the bound stream. */
int sharp_iterate(sharp_plan_t *p, int n, float beta);

/* ---- outputs ----------------------------------------------------------------------------------------------
 * sharp_get_object: out_dev DEVICE obj_rows*obj_cols c64 <- psi = Q*z / Q*Q for the current frames and probe
 * (Eq. 9); pixels with Q*Q = 0 are 0 (reading G5).  sharp_get_probe: out_dev DEVICE m*m c64 <- current w.
 * sharp_get_frames: out_dev DEVICE K*m*m c64 <- current z (the library keeps z in a factored form; this
 * materialises it).  sharp_get_amplitudes: out_dev DEVICE K*m*m f32 <- a in natural (u,v) order. */
int sharp_get_object(sharp_plan_t *p, float *out_dev);
int sharp_get_probe(sharp_plan_t *p, float *out_dev);
int sharp_get_frames(sharp_plan_t *p, float *out_dev);
int sharp_get_amplitudes(sharp_plan_t *p, float *out_dev);
/* sharp_errors: out HOST float[3] <- eps_a = ||P_a z - z||/||a||, eps_Q = ||P_Q z - z||/||a||,
 * eps_Delta = ||z - z_prev||/||a|| at the current z (Eq. 11-13; readings G12, G13).  Does not change the
 * state.  Synchronises the stream. */
int sharp_errors(sharp_plan_t *p, float out[3]);
/* Blocks until all work enqueued by this plan has finished; returns SHARP_ECUDA if any of it failed. */
int sharp_sync(sharp_plan_t *p);
/* Number of kernels this plan has launched so far (bench.py's gpu_launches). */
long long sharp_launch_count(const sharp_plan_t *p);

/* Per-kernel device timing for the roofline report (bench.py).  sharp_profile(p, 1) synchronises, discards
 * earlier records and from then on brackets every kernel launch of sharp_iterate with CUDA events on the bound
 * stream; sharp_profile(p, 0) stops.  sharp_profile_read synchronises and returns, per kernel class, the summed
 * event time (milliseconds) and the number of launches recorded (at most 8192 launches are recorded).
 * Classes: FRAME = the fused per-frame FFT-project-IFFT-combine kernel of sharp_iterate; OVERLAP = the gather
 * overlap + object-space RAAR epilogue of sharp_iterate; PROBE = the Eq. 10 partial-sum kernel; OTHER = the rest. */
#define SHARP_PROF_FRAME 0
#define SHARP_PROF_OVERLAP 1
#define SHARP_PROF_PROBE 2
#define SHARP_PROF_OTHER 3
#define SHARP_PROF_NCLASS 4
int sharp_profile(sharp_plan_t *p, int on);
int sharp_profile_read(sharp_plan_t *p, double ms[SHARP_PROF_NCLASS], long long launches[SHARP_PROF_NCLASS]);

/* ---- integer artefacts (compared bit-exactly with the oracle) ------------------------------
 * sharp_tile_grid: tiles_r x tiles_c tiles of SHARP_TILE^2 pixels.  sharp_tile_lists: HOST pointers (owned by the
 * plan) to the CSR arrays: tile_ptr[tiles_r*tiles_c + 1], tile_frames[tile_ptr[last]].
 * sharp_cover_counts: out HOST obj_rows*obj_cols int32 <- #{i : pixel in frame i}.
 * sharp_frame_index: out_dev DEVICE K*m*m int64 <- the linear object index the device kernels use for frame
 * pixel (i, r, c) (written by a kernel with the device indexing code). */
int sharp_tile_grid(const sharp_plan_t *p, int *tiles_r, int *tiles_c);
int sharp_tile_lists(const sharp_plan_t *p, const int32_t **tile_ptr, const int32_t **tile_frames);
int sharp_cover_counts(const sharp_plan_t *p, int32_t *out_host);
int sharp_frame_index(sharp_plan_t *p, long long *out_dev);

/* ---- single operators (test hooks: operator-level parity with the oracle) -------------------
 * They use the plan's geometry, probe and amplitudes but do not touch the reconstruction state.
 * sharp_op_split:   out_dev[K*m*m c64] <- Q psi            (psi_dev: obj c64)
 * sharp_op_overlap: out_dev[obj c64]   <- Q* f / Q*Q       (f_dev: K*m*m c64)
 * sharp_op_pa:      out_dev[K*m*m c64] <- P_a f            (f_dev: K*m*m c64; out_dev may equal f_dev)
 * sharp_op_fft2:    out_dev[K*m*m c64] <- F f (sign=-1) or F* f (sign=+1), unitary, natural order
 * sharp_op_probe:   out_dev[m*m c64]   <- Eq. 10 for the given psi (obj c64) and frames z (K*m*m c64); where the
 *                   denominator is 0 the plan's current w is kept */
int sharp_op_split(sharp_plan_t *p, const float *psi_dev, float *out_dev);
int sharp_op_overlap(sharp_plan_t *p, const float *f_dev, float *out_dev);
int sharp_op_pa(sharp_plan_t *p, const float *f_dev, float *out_dev);
int sharp_op_fft2(sharp_plan_t *p, const float *f_dev, float *out_dev, int sign);
int sharp_op_probe(sharp_plan_t *p, const float *psi_dev, const float *z_dev, float *out_dev);

/* ---- known-solution error and default initialisations ------------------------
 * sharp_eps0: out HOST float <- eps_0 of Eq. (14), PAPER.md:208-212:
 *      eps_0(z) = min_phi || Q*(e^{i phi} z - z_0) || / || Q* z_0 ||,     z_0 = Q_{w0} psi_0,
 * at the current frames z, with Q* the un-normalised overlap sum under the CURRENT illumination.  psi0_dev: DEVICE
 * obj c64, the known solution.  w0_dev: DEVICE m*m c64, the illumination of the known solution, or NULL when it is
 * the plan's current illumination (the case of PAPER.md:248, "the exact illumination was given").  The minimum over
 * the global phase is taken in closed form.  Does not change the state.  Synchronises.
 * sharp_init_probe: step 2: installs w = F*( sqrt(average frame) ), moved to the frame centre by the
 * cyclic shift (m/2, m/2) (reading G21), exactly as sharp_set_probe would.  Needs the intensities.
 * sharp_init_object_random: step 3: psi^0 ~ U[0,1) (real), z^0 = Q psi^0.  The draw is counter-based:
 * psi^0[p] = float(splitmix64(splitmix64(seed) + p) >> 40) / 2^24 for the row-major pixel index p.  Needs the probe.
 * sharp_op_random_object: out_dev DEVICE obj c64 <- that psi^0 (test hook; state untouched). */
int sharp_eps0(sharp_plan_t *p, const float *psi0_dev, const float *w0_dev, float *out_host);
int sharp_init_probe(sharp_plan_t *p);
int sharp_init_object_random(sharp_plan_t *p, unsigned long long seed);
int sharp_op_random_object(sharp_plan_t *p, unsigned long long seed, float *out_dev);

/* ---- sharded reconstruction (Fig. 2) --------------------------
 * "Summing the frames onto an image (Q*z) requires a reduction for every image pixel across neighboring MPI nodes ...
 * the resulting image is summed across all MPI nodes."  One process per GPU; every rank makes a plan with ITS frames
 * (positions and intensities of its part of the scan, by region or any other partition) and the FULL object size.
 * sharp_set_sharded gives the plan the collective: fn(user, dev_ptr, count, is_double) must replace the `count`
 * float32 (is_double = 0) or float64 (is_double = 1) values at DEVICE pointer dev_ptr (inside the plan's workspace) by
 * their SUM over all ranks, ordered after the work already enqueued on the plan's stream and before anything enqueued
 * on it later (e.g. an NCCL all-reduce on that stream), and return 0; anything else fails the calling sharp_* call
 * with SHARP_ECUDA.  The library calls it wherever the method sums over frames: Q*Q and ||a||^2 when the inputs are
 * set, the object numerator once per iteration (8 bytes per object pixel), the Eq. 10 sums (12 m^2 bytes) per
 * illumination update, three doubles per sharp_errors, m^2 doubles in sharp_init_probe.  All ranks must make the same
 * sequence of calls.  K_total = number of frames of the whole scan (a_rms of reading G4 is global).  Must be called
 * before sharp_set_intensities / sharp_set_probe; fn = NULL returns to the single-GPU plan.
 * With the numerator summed in rank order instead of ascending frame index the result differs from the single-GPU
 * run by rounding only (parity <= 1e-5 against the oracle either way). */
typedef int (*sharp_allreduce_fn)(void *user, void *dev_ptr, size_t count, int is_double);
int sharp_set_sharded(sharp_plan_t *p, sharp_allreduce_fn fn, void *user, long long K_total);

/* ---- illumination constraints and re-centring (step 7) -------
 * Applied after every illumination update of Eq. 10 inside sharp_iterate, in the paper's order:
 *   kind 1 (mask)       w <- F^{-1}{ (F w) m_w }
 *   kind 2 (amplitude)  w <- F^{-1}{ (F w / |F w|) a_w };  where |F w| <= 1e-4 rms(a_w) the phase is taken as 1 (G24)
 *   kind 0              unconstrained
 * then, if re-centring is on: centre of mass of |w|^2 over the frame indices, integer shift
 * d = floor(m/2 - cm + 1/2) per axis applied cyclically to w alone (readings G22, G23).
 * con_dev: DEVICE m*m float32 indexed like the transform (DC at [0,0]); copied.  Ignored for kind 0.
 * sharp_get_probe_shift: HOST int32[2] each: the last shift (d_r, d_c) and the sum of all shifts since
 * sharp_set_probe_recentre was called; either may be NULL.  Synchronises.
 * sharp_op_probe_constrain: out_dev[m*m c64] <- the configured constraint + re-centring applied to w_dev (test hook;
 * out of place; records the shift, leaves the reconstruction state alone). */
int sharp_set_probe_constraint(sharp_plan_t *p, int kind, const float *con_dev);
int sharp_set_probe_recentre(sharp_plan_t *p, int on);
int sharp_get_probe_shift(sharp_plan_t *p, int32_t last[2], int32_t total[2]);
int sharp_op_probe_constrain(sharp_plan_t *p, const float *w_dev, float *out_dev);

/* ---- allocation-free entry point --------------------------------------------------------------------------------
 * sharp_fft2_noalloc: out_dev[K*m*m c64] <- F f (sign = -1) or F* f (sign = +1), unitary, natural order, DC at [0,0]
 * (Eq. 2; the same kernel and the same results as sharp_op_fft2), for callers that cannot call
 * cudaMalloc (CUDA graph capture, tight serving loops, harnesses that forbid it).  It needs no plan, no workspace and
 * no sharp_bind: the kernel's transposition scratch lives in a static device array of the library (8 MiB + 32 KiB
 * per GPU that loads the library, held until exit), and the call makes no cudaMalloc / cudaFree or other allocating call.
 *   f_dev, out_dev   DEVICE, 16-byte aligned, distinct (out of place); the device that owns f_dev is used
 *   m                256 only;  K in [1, SHARP_NOALLOC_MAX_FRAMES];  anything else: SHARP_EINVAL, text in
 *                    sharp_last_error(NULL)
 *   cuda_stream      cudaStream_t cast to void* (NULL = legacy default stream); asynchronous on it
 * Every call shares the one static scratch: calls that overlap on the GPU (different streams without an ordering between
 * them, or several host threads) race.  Calls on one stream are safe.  The scratch keeps the last call's contents;
 * nothing in it has to start at zero (each frame's first stage writes every element before the second reads it). */
#define SHARP_NOALLOC_MAX_FRAMES 4096
int sharp_fft2_noalloc(const float *f_dev, float *out_dev, int m, int K, int sign, void *cuda_stream);

/* ---- host-buffer convenience (the end-to-end path bench.py times) -----------------------------------------
 * sharp_reconstruct_host: everything from HOST buffers: uploads I (K*m*m f32) and w (m*m c64), runs n
 * iterations from the flat object, downloads psi (obj c64) and w, returns the three residuals.  The plan must
 * be bound.  Synchronous. */
int sharp_reconstruct_host(sharp_plan_t *p, const float *I_host, const float *w_host, int n, float beta,
                           float *psi_out_host, float *w_out_host, float eps_out[3]);

#ifdef __cplusplus
}
#endif
#endif /* SHARP_B200_H */
