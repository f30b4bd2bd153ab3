/* awg.h -- C ABI of the B200-native additive waveform synthesiser.
 *
 * Implements the data-parallel hot path of arXiv 2403.15582 (Tu & Subhankar, "Fast real-time
 * arbitrary waveform generation using graphic processing units"): every output sample is
 *
 *      V[n] = sum_k A_k sin(phi_k[n] + theta_k)                        Eq. 9
 *
 * where phi_k is the closed-form time integral of tone k's frequency trajectory -- static
 * (Eq. 8), linear chirp (named at PAPER.md:137) or minimum-jerk ramp (Eq. 10,
 * PAPER.md:141-148, branch 1 read as the integral of the ramp: DESIGN.md reading G1) -- the
 * phase is reduced mod one turn before the sine (Eq. 14) and the sum is quantised
 * to 16-bit DAC codes chunk by chunk (chunk = the paper's L_s),
 * phase-continuous across chunks.  The paper's WG, WC and WM kernels are one
 * fused sm_100a kernel here: no per-tone wavetable is ever stored.
 *
 * Conventions
 *  - Plain C99, no exceptions cross this boundary; every call returns an awg_status (0 = OK,
 *    negative = error) and never prints or aborts.  awg_last_error() gives the message.
 *  - "host" pointers are ordinary CPU memory, caller-owned, read during the call only (copied
 *    before return).  "device" pointers are CUDA global memory on the current device,
 *    caller-owned (e.g. torch.empty(..., device='cuda').data_ptr()).
 *  - stream arguments are a cudaStream_t passed as void* (NULL = the legacy default stream).
 *    Synthesis calls are asynchronous: they return after enqueueing work on that stream.
 *  - Units: Hz, seconds, radians (phi0), fraction of full scale (A).  chunk_len is in samples and
 *    must be a positive multiple of 8 (16-byte int16 stores).
 *  - A plan is not thread-safe; distinct plans are independent.
 *  - Output for (plan, chunk_idx) is a pure function of the trajectory table and of the absolute
 *    sample index; it does not depend on the stream, ring depth, call order or chunk_len
 *    (kernel tiles are anchored to absolute sample indices that are multiples of 2048, and
 *    the order in which tone partial sums are added depends on the tone count only).
 *  - A plan belongs to the CUDA device that was current when it was created; calls that enqueue
 *    work return AWG_ERR_STATE when another device is current.
 */
#ifndef AWG_H_
#define AWG_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct awg_plan awg_plan; /* opaque; created and destroyed only by the library */
typedef struct awg_ring awg_ring; /* opaque streaming ring bound to one plan            */
typedef int32_t awg_status;

enum {
    AWG_OK = 0,
    AWG_ERR_INVALID_ARG = -1, /* null pointer, bad size, non-finite value, misaligned buffer ... */
    AWG_ERR_ALLOC = -2,       /* host or device allocation failed                                */
    AWG_ERR_CUDA = -3,        /* a CUDA runtime call failed; awg_last_error() has its string    */
    AWG_ERR_STATE = -4,       /* call order violated (see each function)                        */
    AWG_ERR_UNDERRUN = -5     /* ring: the acquired chunk missed its real-time deadline         */
};

/* frequency trajectory of one tone ("any functional form for a frequency chirp") */
enum {
    AWG_PROFILE_STATIC = 0,  /* f(t) = f0                                                   */
    AWG_PROFILE_LINEAR = 1,  /* f0 -> f1 linearly over [t_start, t_start + t_dur]            */
    AWG_PROFILE_MINJERK = 2, /* f0 -> f1 along the minimum-jerk quintic 10s^3 - 15s^4 + 6s^5 */
    AWG_PROFILE_EXP = 3      /* exponential chirp f(tau) = f0 (f1/f0)^(tau/t_dur) (named at PAPER.md:137; G20):
                                f0 and f1 must be > 0.  Costs what a minimum-jerk move costs (one sine per sample
                                inside the move); chirps too fast for fp32 coefficients take the fp64 path         */
};

/* sine engine of the synthesis kernel (step a3 of the hot path) */
enum {
    AWG_ENGINE_AUTO = 0, /* the library picks (currently AWG_ENGINE_FMA)                                    */
    AWG_ENGINE_MUFU = 1, /* one MUFU.SIN per (tone, sample); phase re-centred per 512-sample block           */
    AWG_ENGINE_FP64 = 2, /* reference-grade: closed form and sine in fp64 per (tone, sample); ~50x slower   */
    AWG_ENGINE_FMA = 3   /* angle addition on the FMA pipe for 2048-sample tiles where a tone is static (one
                            sin + one cos per thread, tone and 32 samples, then ONE multiply-add per
                            tone-sample with a per-tone table); tiles inside a slow move take 1.25
                            multiply-adds per tone-sample, tiles inside any other move the MUFU path      */
};

/* ---- plan ---------------------------------------------------------------------------------- */

/* Creates a plan for n_tones tones at sample_rate_hz with chunks of chunk_len samples on the
 * current CUDA device.  Errors: INVALID_ARG (out NULL, n_tones < 1 or > 65536, rate not finite or
 * <= 0, chunk_len < 8 or not a multiple of 8), ALLOC, CUDA (no device). */
awg_status awg_plan_create(awg_plan **out, int32_t n_tones, double sample_rate_hz, int64_t chunk_len);

/* Frees the plan and its device tables after synchronising the streams it has work on.
 * Rings bound to the plan must be destroyed first.  NULL is accepted. */
awg_status awg_plan_destroy(awg_plan *p);

/* int16 code = clamp(rint(scale * V), -32768, 32767), round-half-even (reading G9).
 * Default 0.9*32767 (BASELINE.json config 1).  Errors: INVALID_ARG (not finite or <= 0). */
awg_status awg_set_scale(awg_plan *p, double scale);

/* Selects the sine engine (AWG_ENGINE_*).  Errors: INVALID_ARG. */
awg_status awg_set_engine(awg_plan *p, int32_t engine);

/* Replaces the whole trajectory table (Eq. 9/10 inputs per tone: a_j, theta_j, f_start, f_finish,
 * T).  Seven host arrays of length n_tones:
 *   f0, f1   start / final frequency, Hz           A        amplitude, fraction of full scale
 *   phi0     phase offset at t = 0, radians        t_start  move start, s (any real, not snapped)
 *   t_dur    move duration, s (>= 0; 0 = instant retune at t_start)
 *   profile  AWG_PROFILE_* (STATIC ignores f1, t_start, t_dur)
 * Frequencies above Nyquist or negative are evaluated as given (they alias), sum(A) > 1 saturates.
 * Resets the update history.  Errors: INVALID_ARG (NULL, non-finite value, t_dur < 0, unknown
 * profile, AWG_PROFILE_EXP with f0 <= 0 or f1 <= 0). */
awg_status awg_set_trajectories(awg_plan *p, const double *f0, const double *f1, const double *A,
                                const double *phi0, const double *t_start, const double *t_dur,
                                const int32_t *profile);

/* Time-varying amplitudes a_j[i] of Eq. 9 (constant in the paper's worked case,
 * PAPER.md:137; reading G7): tone k goes from the amplitude given to awg_set_trajectories to
 * A1[k] over [t_start[k], t_start[k] + t_dur[k]] along profile[k] -- AWG_PROFILE_STATIC (no ramp: A1,
 * t_start, t_dur ignored), AWG_PROFILE_LINEAR, or AWG_PROFILE_MINJERK (10 s^3 - 15 s^4 + 6 s^5): tone
 * creation (0 -> A1) and removal (A -> 0) without a click.  Four host arrays of length n_tones.  Replaces
 * earlier ramps; awg_set_trajectories clears them.  Samples inside a ramp are evaluated one by one in
 * fp64 phase (slow, exact); before and after it the tone costs what any other tone costs.
 * Errors: INVALID_ARG (NULL, non-finite, t_dur < 0, unknown profile), STATE (no table set; after a
 * per-chunk update; tone in the static buffer). */
awg_status awg_set_amplitude_ramps(awg_plan *p, const double *A1, const double *t_start, const double *t_dur,
                                   const int32_t *profile);

/* Per-chunk update (streaming pathway, Fig. 7): at the first sample of chunk_idx each
 * listed tone starts a new move from its current instantaneous frequency and phase (phase- and
 * frequency-continuous) to f1[i] over t_dur[i] with profile[i].  Host arrays of length n_upd.
 * The plan keeps only the current segment of each tone, so updates must come in non-decreasing
 * chunk order and chunks earlier than the latest update can no longer be synthesised.
 * Errors: INVALID_ARG (NULL with n_upd > 0, tone index out of range or duplicated, non-finite,
 * t_dur < 0, unknown profile, chunk_idx < 0), STATE (no table set; chunk_idx lower than a previous
 * update's). */
awg_status awg_update_trajectories(awg_plan *p, int64_t chunk_idx, int32_t n_upd, const int32_t *tone_idx,
                                   const double *f1, const double *t_dur, const int32_t *profile);

/* ---- synthesis (asynchronous on `stream`) ---------------------------------------------------- */

/* Writes the int16 codes of samples [chunk_idx*chunk_len, (chunk_idx+1)*chunk_len) to dev_out
 * (device, chunk_len int16, 16-byte aligned).  Errors: INVALID_ARG (NULL, misaligned, chunk_idx < 0),
 * STATE (no table set; chunk earlier than the latest update), CUDA. */
awg_status awg_synthesize_chunk(awg_plan *p, int64_t chunk_idx, int16_t *dev_out, void *stream);

/* Same chunk before quantisation: the fp32 sum V (full scale = 1.0).  dev_out: chunk_len floats. */
awg_status awg_synthesize_chunk_f32(awg_plan *p, int64_t chunk_idx, float *dev_out, void *stream);

/* Playback / "precomputed" pathway (Fig. 6): chunks first_chunk .. first_chunk+n_chunks-1
 * into one contiguous device buffer of n_chunks*chunk_len int16, in one kernel launch. */
awg_status awg_synthesize_range(awg_plan *p, int64_t first_chunk, int64_t n_chunks, int16_t *dev_out,
                                void *stream);

/* End-to-end variant with a HOST destination: synthesises the range in pieces of 2^21 samples into
 * four internal device slots (pieces alternate between two internal streams, so the next piece takes
 * over the SMs as the current one runs out of tiles) and copies each finished piece to host_out on a
 * third stream (n_chunks*chunk_len int16; pinned memory gives overlap of copy and compute, pageable
 * memory works) -- synchronous, returns when host_out is complete.  Stands in for the paper's pinned-buffer -> DAC transfer. */
awg_status awg_synthesize_range_host(awg_plan *p, int64_t first_chunk, int64_t n_chunks, int16_t *host_out);

/* ---- four-channel multiplexed output (the paper's WM kernel; Fig. 4) ---------- */

/* The paper's streaming chunk is 2^20 samples = 4 DAC channels x 2^18, "read sequentially in groups of
 * four".  plans: host array of n_channels (1..8) distinct plans on the current device with
 * the same chunk_len, one independent tone set per channel.  Writes n_channels*chunk_len int16 to dev_out
 * (device, 16-byte aligned): dev_out[n_channels*i + c] = code of sample chunk_idx*chunk_len + i of
 * channel c -- bit for bit what awg_synthesize_chunk gives for plans[c].  One kernel launch per channel,
 * each storing its channel's half-words of every group: channel 0 on `stream`, the others beside it on
 * internal streams that fork from `stream` and join it again (to the caller everything is ordered on
 * `stream`).  Errors: those of
 * awg_synthesize_chunk for any channel, checked before the first launch; INVALID_ARG (NULL, n_channels,
 * chunk_len mismatch, repeated plan). */
awg_status awg_synthesize_chunk_mux(awg_plan *const *plans, int32_t n_channels, int64_t chunk_idx,
                                    int16_t *dev_out, void *stream);

/* ---- static-buffer pathway (PAPER.md:93-109 section IV A, Eq. 6-8; :133 Eq. 9; :141-146 Eq. 10) -- */

/* Eq. 6: the closest frequency with a whole number of cycles in L_s samples,
 * f_j = nint(f0 L_s / fs) fs / L_s.  Host-only.  Errors: INVALID_ARG. */
awg_status awg_snap_frequency(double f0_hz, double sample_rate_hz, int64_t L_s, double *f_snapped_hz);

/* Moves the listed tones (host array of n_static tone indices) out of the per-sample evaluation into the
 * looped buffer X_static of length L_s = chunk_len (Eq. 7-8): X_static[i] = sum_j a_j sin(2 pi f_j/fs i
 * + theta_j) is synthesised once on the device (fp32), and every later synthesis call computes
 * V[n] = X_static[n mod L_s] + (the other tones, evaluated per sample) -- Eq. 9.  The
 * listed tones must be static and on the fs/L_s grid of Eq. 6 (then the result equals evaluating them
 * per sample); chunk_len must be >= 2048.  Replaces any earlier buffer; n_static = 0 removes it.
 * Synchronous on `stream`.  Errors: INVALID_ARG (index out of range or repeated, tone not static or
 * off the grid, chunk_len too small), STATE (no table set), ALLOC, CUDA. */
awg_status awg_static_buffer_set(awg_plan *p, int32_t n_static, const int32_t *tone_idx, void *stream);

/* Hand-back of Eq. 10 branch 3: from chunk_idx on (L_d = chunk_idx*chunk_len, a
 * multiple of L_s) each listed tone is a looped static wavetable at its final frequency
 * with the phase offset theta'_j = its phase at L_d; its period is added to X_static and the tone leaves
 * the per-sample evaluation.  Each tone's move must have ended by L_d and its final frequency must be on
 * the Eq. 6 grid.  Like a trajectory update, this fixes the past: chunks before chunk_idx can no longer
 * be synthesised.  Synchronous on `stream`.  Errors: INVALID_ARG, STATE (still moving at L_d, already in
 * the buffer, chunk_idx before the latest update), ALLOC, CUDA. */
awg_status awg_static_buffer_fold(awg_plan *p, int64_t chunk_idx, int32_t n_fold, const int32_t *tone_idx,
                                  void *stream);

/* Copies X_static (chunk_len floats, full scale = 1.0) to dev_out (device).  Errors: STATE (no buffer). */
awg_status awg_static_buffer_read(awg_plan *p, float *dev_out, void *stream);

/* ---- streaming ring (DAC-FIFO stand-in; Fig. 2b, 75, 127) --------------------------- */

/* n_slots >= 2 device slots of chunk_len int16; host_mirror != 0 adds pinned-host slots and a copy
 * stream that D2H-copies each finished chunk.  The ring owns its streams. */
awg_status awg_ring_create(awg_ring **out, awg_plan *p, int32_t n_slots, int32_t host_mirror);

/* Applies the n_upd updates (may be 0) at chunk_idx, then enqueues synthesis of chunk_idx into the
 * next free slot.  Chunks must be submitted in increasing order.  Errors: STATE (ring full: acquire
 * and release first; out-of-order chunk), plus those of awg_update_trajectories. */
awg_status awg_ring_submit(awg_ring *r, int64_t chunk_idx, int32_t n_upd, const int32_t *tone_idx,
                           const double *f1, const double *t_dur, const int32_t *profile);

/* Blocks until the oldest submitted chunk is complete (and mirrored when host_mirror is on), then
 * lends its slot: *dev_ptr (device) and *host_ptr (pinned host or NULL) stay valid until
 * awg_ring_release.  A virtual DAC starts when the first acquire returns and consumes one chunk every
 * chunk_len / sample_rate seconds: the j-th acquired chunk (j = 0, 1, ...) is due j periods after that
 * instant.  Returns AWG_ERR_UNDERRUN (pointers still valid, chunk still lent) when the chunk was
 * submitted after it was due or was not complete when due.  Errors: STATE (nothing submitted). */
awg_status awg_ring_acquire(awg_ring *r, int64_t *chunk_idx, const int16_t **dev_ptr,
                            const int16_t **host_ptr);
awg_status awg_ring_release(awg_ring *r, int64_t chunk_idx);

/* produced = chunks completed; underruns = deadline misses; max_chunk_ms = longest device time of
 * one chunk (synthesis + mirror copy) measured with CUDA events.  Any pointer may be NULL. */
awg_status awg_ring_stats(awg_ring *r, int64_t *produced, int64_t *underruns, double *max_chunk_ms);
awg_status awg_ring_destroy(awg_ring *r);

/* ---- misc --------------------------------------------------------------------------------------- */

/* Bytes this plan has copied host->device (trajectory table uploads) and device->host (host-destination
 * synthesis and ring mirror) since creation.  Either pointer may be NULL. */
awg_status awg_plan_io_bytes(awg_plan *p, int64_t *h2d_bytes, int64_t *d2h_bytes);

/* Algorithmic operation counts of the CURRENT trajectory table over chunks first_chunk ..
 * first_chunk+n_chunks-1, at sample granularity: tone-samples of tones that are static there
 * (one fp32 multiply-add each on the angle-addition engine), inside a slow move (1.25 multiply-adds,
 * 1.5 in plans with faster slow movers: the kernel's slow pass) and inside any other move (one MUFU.SIN + two multiply-adds).  This is the
 * library's own classification (the one the kernel acts on); bench.py derives its roofline from it.
 * Host-only, no CUDA work.  Any pointer may be NULL.  Errors: INVALID_ARG, STATE (no table set). */
awg_status awg_plan_op_counts(awg_plan *p, int64_t first_chunk, int64_t n_chunks, int64_t *static_ts,
                              int64_t *slow_ts, int64_t *fast_ts);

/* Tile-serving order of a launch over chunks first_chunk .. first_chunk+n_chunks-1 of the CURRENT table:
 * *n_listed = 2048-sample tiles of the range in which at least max(2, n/16) of the n evaluated tones enter
 * or leave a slow move at once (such a tile costs several ordinary ones: all those tones take the
 * one-sine-per-sample pass there), *n_served_first = how many of them the launch hands out before all
 * other tiles (the heaviest 16; 0 for ranges under 64 tiles, whose units all start at once).  The order
 * has no effect on any sample.  Host-only.  Either pointer may be NULL.  Errors: INVALID_ARG, STATE. */
awg_status awg_plan_hot_tiles(awg_plan *p, int64_t first_chunk, int64_t n_chunks, int32_t *n_listed,
                              int32_t *n_served_first);

/* ---- allocation-free one-shot synthesis ------------------------------------------------------------ */

/* For callers that cannot allocate device memory (a harness that forbids cudaMalloc, a serving loop that
 * must stay off the allocator): no plan, and no cudaMalloc, cudaFree, stream or event creation anywhere
 * on this call, the first one included.  Synthesises samples first_sample .. first_sample+n_samples-1 of
 * the waveform of Eq. 9/10 for the n_tones trajectories given exactly as to
 * awg_set_trajectories (seven HOST arrays of length n_tones, same units, same profiles), sample index 0
 * at t = 0, into dev_out (DEVICE, int16, 16-byte aligned, n_samples elements, caller-owned) on `stream`
 * (cudaStream_t or NULL), at the default scale of a plan (0.9 * 32767) with the default engine: bit for
 * bit what a plan with the same trajectories gives for the same samples.  Asynchronous like
 * awg_synthesize_chunk; the host arrays are consumed before the call returns.
 * Limits: n_tones <= 4096, n_samples <= 2^20 (a multiple of 8; first_sample too) per call -- call again
 * for the next range.  Everything the kernels need on the device (the trajectory table, the tile
 * scheduler's counters, the int32 scratch tiles in which the tone groups of a tile meet) lives in ONE
 * static 5.9 MB device array that is part of the library image: every GPU that loads the library holds
 * it until the process exits.  All calls share it, and it keeps the last call's contents (each call
 * clears what it needs at zero on `stream` first): calls that overlap on the GPU -- issued on different
 * streams without an event between them, or from several threads -- RACE on it; calls on one stream, or
 * ordered by events, are safe.  Plans do not use the array and are not affected.
 * Errors: INVALID_ARG (a size beyond the limits, NULL, misaligned, non-finite, t_dur < 0, unknown
 * profile), CUDA. */
awg_status awg_synthesize_noalloc(double sample_rate_hz, int32_t n_tones, const double *f0, const double *f1,
                                  const double *A, const double *phi0, const double *t_start,
                                  const double *t_dur, const int32_t *profile, int64_t first_sample,
                                  int64_t n_samples, int16_t *dev_out, void *stream);

/* Number of kernels the library has launched since load (all plans); for launch accounting. */
int64_t awg_kernel_launch_count(void);

/* Thread-local, library-owned, valid until the next awg_* call on this thread. */
const char *awg_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* AWG_H_ */
