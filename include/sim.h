/*
 * sim.h -- C ABI of the B200 fast-mode radar raw-data library (libsim.so).
 *
 * Method: "fast simulation mode" of Monnier, Camus, Hellouvry, arxiv 2408.11472 (section III).
 * Every `n_fast` pulses the scene is evaluated once; each illuminated scatterer is summed into a
 * per-update [range gate x Doppler bin] spectrum (Algorithm 1 + `rasterize`); the
 * spectra are turned into long-time signals by inverse 1-D DFTs along Doppler and
 * neighbouring updates are combined with the weights of eq. (1).
 * The readings taken where the paper is silent are listed in DESIGN.md ("Readings").
 *
 * Conventions
 *   - Plain C types only.  Every pointer says whether it is a HOST or a DEVICE pointer.
 *   - Frame: local Cartesian, z up, flat Earth.  Scatterer arrays are fp32, satellite state fp64.
 *   - The library never allocates device memory: the caller passes one workspace
 *     (sim_workspace_bytes) that must outlive the handle.  The library owns only the host handle,
 *     and (when host staging is enabled) one internal copy stream and a few events.
 *   - Every call enqueues work on the CUDA stream given to sim_create and returns without
 *     synchronising, unless stated.  Device inputs must stay valid until the stream reaches that point.
 *     Stream order holds for them: whatever was enqueued earlier on that stream (a kernel of the caller's that writes
 *     the scatterer arrays, say) is complete and visible before a kernel of the library reads them.
 *   - Every function returns SIM_OK or a negative SIM_ERR_*; nothing throws, nothing aborts.  After
 *     an error the handle is unchanged and still usable.  sim_last_error gives a message.
 *   - Not thread-safe per handle.  Distinct handles are independent.
 */
#ifndef PAPER_2408_11472_SIM_H
#define PAPER_2408_11472_SIM_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define SIM_OK 0
#define SIM_ERR_INVALID_ARG (-1) /* NULL pointer, negative count, misaligned array, bad flag */
#define SIM_ERR_BAD_CONFIG (-2)  /* sizes out of range, N with a prime factor other than 2, 3, 5, non-positive lambda/PRF/dR */
#define SIM_ERR_WORKSPACE (-3)   /* workspace too small or not 256-byte aligned */
#define SIM_ERR_NOT_READY (-4)   /* synthesis needs a spectrum that has not been accumulated */
#define SIM_ERR_OVERFLOW (-5)    /* more pending spectra than max_pending_updates */
#define SIM_ERR_CUDA (-6)        /* a CUDA runtime call failed (message in sim_last_error) */

#define SIM_W_SQRT 0   /* eq. (1) of the paper: W = (1 - |i-x|/n_fast)^(1/2); sum of squares = 1 */
#define SIM_W_LINEAR 1 /* W = 1 - |i-x|/n_fast; partition of unity (reading A1) */

#define SIM_ACC_APPEND 1u /* sim_accumulate_update: add to the current update instead of starting one */
#define SIM_SYN_FINAL 1u  /* sim_synthesize_pulses: a missing successor spectrum is allowed (tail rule) */

/* Doppler source of step A4.
 *   SIM_DOPPLER_ANALYTIC:   f_D = -2 (v_p - v_sat).u / lambda  (north_star; reading A5).
 *   SIM_DOPPLER_PULSE_PAIR: the paper's estimator, Algorithm 1 lines 5-7: the scene one
 *     PRI later (scatterers and satellite moved by v / PRF), D = arg(C_{i+1} C_i^*) PRF / 2 pi
 *     = -2 (R' - R) PRF / lambda, aliased into the N bins (readings A6, R4). */
#define SIM_DOPPLER_ANALYTIC 0
#define SIM_DOPPLER_PULSE_PAIR 1

#define SIM_GATE_NONE INT32_MIN /* sim_debug_indices: scatterer touches no gate / is dropped */

typedef struct sim_handle sim_handle; /* opaque, host memory, owned by the library */

typedef struct sim_config {
  uint32_t struct_size;        /* = sizeof(sim_config); ABI guard */
  int32_t n_gates;             /* G = n_range of T_fast, 1..1024 */
  int32_t n_doppler;           /* N = n_doppler of T_fast, 16..4096 with no prime factor other than 2, 3 and 5 (mixed-radix
                                  inverse FFT): the paper's n_fast = 250 ... 1250 run exactly as N = P, or
                                  as N = 2P, which keeps the past and the future half of a long signal apart (A4) */
  int32_t pulses_per_update;   /* P = n_fast, >= 1 */
  int32_t max_pending_updates; /* spectra kept in the ring, >= 2 */
  int32_t weight_mode;         /* SIM_W_SQRT (default, the paper) or SIM_W_LINEAR */
  int32_t device;              /* CUDA device ordinal the workspace and stream live on */
  int32_t doppler_mode;        /* SIM_DOPPLER_ANALYTIC (default) or SIM_DOPPLER_PULSE_PAIR */
  double wavelength_m;         /* lambda > 0 */
  double prf_hz;               /* PRF > 0 */
  double gate_spacing_m;       /* Delta R > 0 */
  double antenna_alpha;        /* G(theta) = exp(-alpha sin^2 theta) >= 0; 0 = isotropic (reading A10) */
  int64_t host_stage_scatterers; /* 0, or the H2D chunk size (scatterers) of the *_host entry points */
  int64_t host_stage_pulses;     /* 0, or the most pulses one sim_synthesize_pulses_host call may ask */
} sim_config;

/* One batch of scatterers, struct-of-arrays, n entries each (the paper's facets of one tile,
 * PAPER.md:39).  Pointers are DEVICE pointers for sim_accumulate_update / sim_debug_indices and
 * HOST pointers (pinned memory for copy/compute overlap) for sim_accumulate_update_host.
 * Device arrays must be 16-byte aligned.  s0dA = sigma0 * dA (NRCS times facet area, m^2). */
typedef struct sim_scatterers {
  const float *x, *y, *z;    /* position, m */
  const float *vx, *vy, *vz; /* velocity, m/s */
  const float *s0dA;         /* <= 0 or NaN: the scatterer contributes nothing */
  uint64_t n;
} sim_scatterers;

/* Satellite state at the update instant t_u = u * P / PRF; HOST struct, read during
 * the call. */
typedef struct sim_sat_state {
  double pos[3];        /* m */
  double vel[3];        /* m/s */
  double boresight[3];  /* antenna axis, any non-zero vector (normalised by the library) */
  double range_gate0_m; /* range of the centre of gate 0 (reading A9) */
} sim_sat_state;

typedef struct sim_stats {
  uint64_t kernel_launches;      /* kernels of this library launched since sim_create */
  uint64_t updates_accumulated;  /* spectra started */
  uint64_t scatterers_seen;      /* scatterers passed to sim_accumulate_update[_host] */
  int64_t pulses_emitted;        /* pulses written by sim_synthesize_pulses[_host] */
} sim_stats;

/* Bytes of DEVICE workspace sim_create needs for this configuration.  HOST pointers. */
int sim_workspace_bytes(const sim_config* cfg, size_t* out_bytes);

/* Create a handle.  d_workspace: DEVICE pointer, 256-byte aligned, `bytes` >= sim_workspace_bytes,
 * owned by the caller and kept alive until sim_destroy.  cuda_stream: a cudaStream_t (NULL = the
 * legacy default stream).  Initialises the twiddle table on the stream.  Every call makes cfg.device current for its
 * own duration and restores the caller's current device before it returns. */
int sim_create(const sim_config* cfg, void* d_workspace, size_t bytes, void* cuda_stream,
               sim_handle** out);

/* Steps A1-A7: Algorithm 1 body for one surface update.
 * For every scatterer p: range R = |r_p - r_sat| (scatterers_range), two-gate linear weight from
 * gf = (R - range_gate0)/dR, Doppler bin k = round(f_D N / PRF) mod N with
 * f_D = -2 (v_p - v_sat).u / lambda, complex amplitude
 * sqrt(s0dA) G(theta) / R^2 exp(-i 4 pi R / lambda) (scatterers_complex_amplitudes), summed into the
 * [G][N] complex64 spectrum of the update (rasterize).
 * flags = 0: start update u = (number of updates so far), zero its spectrum, accumulate `scat`.
 * flags = SIM_ACC_APPEND: add another batch (tile) to the update started last.
 * Errors: SIM_ERR_OVERFLOW when the ring is full of spectra synthesis still needs;
 * SIM_ERR_INVALID_ARG for NULL / misaligned arrays, APPEND before any update.  scat->n may be 0. */
int sim_accumulate_update(sim_handle* h, const sim_scatterers* d_scat, const sim_sat_state* sat,
                          uint32_t flags);

/* Steps S1-S3: post-processing.  Emits the next n_pulses pulses of the
 * stream: for pulse x in segment s = floor(x/P),
 *   Y[x][g] = W_s(x) y_s[g][(x - sP) mod N] + W_{s+1}(x) y_{s+1}[g][(x - (s+1)P) mod N],
 * y_u = unnormalised inverse DFT of spectrum u along Doppler, W from eq. (1).
 * d_iq: DEVICE, complex64 [n_pulses][G] (pulse-major, gate fastest, interleaved re/im), 16-byte aligned.
 * Without SIM_SYN_FINAL every segment touched needs spectra s and s+1 (else SIM_ERR_NOT_READY, nothing
 * emitted).  With SIM_SYN_FINAL a segment whose successor is absent uses y_s at weight 1.
 * Spectra older than the segment of the next pulse are released from the ring. */
int sim_synthesize_pulses(sim_handle* h, int64_t n_pulses, void* d_iq, uint32_t flags);

/* Same two calls with HOST buffers (pinned for overlap): the library stages through the workspace
 * (cfg.host_stage_scatterers / host_stage_pulses must be > 0) with double-buffered cudaMemcpyAsync.
 * sim_synthesize_pulses_host enqueues the device-to-host copy on the stream; call sim_synchronize
 * (or synchronise the stream) before reading h_iq. */
int sim_accumulate_update_host(sim_handle* h, const sim_scatterers* h_scat, const sim_sat_state* sat,
                               uint32_t flags);
int sim_synthesize_pulses_host(sim_handle* h, int64_t n_pulses, void* h_iq, uint32_t flags);

/* Blocks until all work enqueued by this handle has finished. */
int sim_synchronize(sim_handle* h);

/* Frees the host handle (and internal stream/events).  NULL-safe.  The workspace stays the caller's. */
int sim_destroy(sim_handle* h);

/* ---- parity / debug / multi-GPU support ------------------------------------------------------ */

/* Copies spectrum `update_index` (must still be in the ring) to d_out: DEVICE complex64 [G][N],
 * bin fastest.  Asynchronous on the stream. */
int sim_get_spectrum(sim_handle* h, int64_t update_index, void* d_out);

/* Byte offset of spectrum `update_index` inside the caller's workspace (so that the caller can
 * all-reduce partial spectra across GPUs in place). */
int sim_spectrum_offset(sim_handle* h, int64_t update_index, size_t* out_offset);

/* REGULAR MODE (reading R5): the at-scale truth the fast mode
 * approximates.  Scatterers (DEVICE arrays) and satellite are in uniform motion from the states given for pulse 0;
 * for each pulse j = first_pulse .. first_pulse + n_pulses - 1 (any sign), at t_j = j / PRF, every scatterer's
 * complex amplitude sqrt(s0dA) G(theta) / R^2 exp(-i 4 pi R / lambda) at ITS RANGE AT t_j is summed into its two
 * gates (the linear split of step A3).  d_iq: DEVICE complex64 [n_pulses][G], gate fastest, 16-byte aligned.
 * flags = 0: d_iq is zeroed first; SIM_ACC_APPEND: the sums are added to it (scenes delivered in pieces).
 * Work is scatterers x pulses.  Independent of the spectra ring and of sim_synthesize_pulses.
 * Errors: SIM_ERR_INVALID_ARG (NULL / misaligned), SIM_ERR_BAD_CONFIG (n_gates > ~830, or a gate window too
 * deep for the polynomial gate coordinate). */
int sim_regular_pulses(sim_handle* h, const sim_scatterers* d_scat, const sim_sat_state* sat,
                       int64_t first_pulse, int64_t n_pulses, void* d_iq, uint32_t flags);

/* Delay-Doppler burst step (reading R8): the IQ stream is split into
 * bursts of `burst` pulses (64 in the paper; a power of two in 16..128) and each burst gets an along-track FFT per
 * gate: beams[b][k][g] = sum_m iq[b burst + m][g] exp(-2 pi i k m / burst), unnormalised, beam k in natural FFT order.
 * d_iq: DEVICE complex64 [n_pulses][G]; d_beams: DEVICE complex64 [n_pulses / burst][burst][G]; out of place; 16-byte
 * aligned; n_pulses a multiple of burst.  The Doppler-centroid and range-migration corrections of the paper need
 * instrument data and are not part of it. */
int sim_burst_beams(sim_handle* h, const void* d_iq, int64_t n_pulses, int32_t burst, void* d_beams, uint32_t flags);

/* Tabulated antenna pattern (section II.A: "all antenna patterns ... are computed and recorded on a u-v
 * grid.  The complex values of all antenna patterns at each facet are then obtained through interpolation in the u-v
 * grid"; reading R9).  With a table set, G(theta) of every later accumulation (fast mode;
 * sim_regular_pulses refuses a table with SIM_ERR_BAD_CONFIG) is the complex value interpolated bilinearly at the direction cosines
 *   u = d.e1 / R,  v = d.e2 / R,   d = r_p - r_sat,
 *   b = unit boresight, e1 = unit vector of v_sat - (v_sat.b) b (along track, normal to b), e2 = b x e1;
 * a direction outside [u0, u0 + (n_u-1) du] x [v0, v0 + (n_v-1) dv] is outside the recorded pattern: gain 0.
 * d_table: DEVICE complex64 [n_v][n_u] (u fastest, interleaved re/im), 8-byte aligned, owned by the caller and kept
 * alive while it is set; n_u, n_v in 2..4096; du, dv > 0.  d_table = NULL: back to the analytic exp(-alpha sin^2 theta).
 * Interpolation runs in fp32: the table should resolve the pattern (relative change per cell well below 1).
 * Errors: SIM_ERR_INVALID_ARG (sizes, steps, alignment).  An accumulation with a table set and a satellite velocity
 * parallel to the boresight returns SIM_ERR_INVALID_ARG (no along-track axis). */
int sim_set_antenna_lut(sim_handle* h, const void* d_table, int32_t n_u, int32_t n_v, double u0, double du, double v0,
                        double dv);

/* Runs the production index computation only: for each scatterer the gate g0 = floor(gf) in
 * [-1, G-1] and the Doppler bin k in [0, N); dropped scatterers give (SIM_GATE_NONE, -1).
 * d_gate0, d_bin: DEVICE int32[n].  Must match the canonical fp64 sequence bit for bit. */
int sim_debug_indices(sim_handle* h, const sim_scatterers* d_scat, const sim_sat_state* sat,
                      int32_t* d_gate0, int32_t* d_bin);

/* Tuning knobs (benchmarks and tests; defaults are chosen by the library). */
#define SIM_OPT_ACC_VARIANT 1   /* 4 = production kernel (default), 0 = reference kernel (one thread per scatterer, canonical
                                   sequence, global fp64 reductions; the A/B partner in the parity tests).
                                   Selecting a variant resets warps / per-lane / epoch options to the defaults */
#define SIM_OPT_ACC_BLOCKS 2    /* grid size of the accumulation kernel; 0 = auto (resident blocks x SMs) */
#define SIM_OPT_ACC_SUPERCHUNK 3 /* scatterers per scheduling unit (rounded up to whole fixed-point epochs); 0 = auto */
#define SIM_OPT_ACC_WINDOW_BINS 4 /* Doppler bins held in shared memory; 0 = auto (as many as fit, up to 20) */
#define SIM_OPT_GUARD_LSB 5     /* guard band of the fast index path in units of 2^-20 gate / bin (default 16) */
#define SIM_OPT_ACC_WARPS 9      /* warps per block: 8 (default, two blocks per SM) or 16 */
#define SIM_OPT_ACC_PER_LANE 11  /* scatterers per lane per chunk: 2 or 4 (default) */
#define SIM_OPT_ACC_EPOCH 12     /* scatterers per fixed-point epoch: 64..16383 (default 8191) */
#define SIM_OPT_ACC_SCATTER 14   /* 1 (default) = scheduling units visit the scene in a scattered order (dark and
                                    illuminated parts in flight together); 0 = in input order */
#define SIM_OPT_ACC_INTERLEAVE 15 /* scatterers in flight per lane at a time: 2 or 4 (<= per lane) */
#define SIM_OPT_ACC_SHAPE 16      /* block shape in one call: (warps << 16) | (per lane << 8) | interleave;
                                     compiled shapes: (8,4,4) default, (8,4,2), (8,2,2), (16,4,4) */
#define SIM_OPT_INDEX_PATH 6    /* 0 = canonical fp64 sequence everywhere, 1 = fast path + guard band (default) */
int sim_set_option(sim_handle* h, int32_t option, int64_t value);

int sim_get_stats(const sim_handle* h, sim_stats* out);

/* Synchronises the stream, copies the library's device counters to h_out (HOST, 4 x uint32) and, when reset != 0,
 * zeroes them.  [1] scatterers whose contributions left the shared-memory tile for global reductions (outside the
 * Doppler window / above the fixed-point range / guard band), [3] scatterers whose indices the canonical sequence
 * decided (guard band); both since the last reset.  [0] and [2] are the accumulation kernel's own scheduling words
 * (ticket counter, blocks finished): each launch leaves them at 0, they carry no information between launches. */
int sim_read_counters(sim_handle* h, uint32_t* h_out, int32_t reset);

/* ---- one update without any device allocation by anybody ------------------------------------------ */

/* Every call above needs a device workspace, and somebody has to allocate it.  Some users of this library cannot:
 * a radar-chain plug-in running inside a host simulator that took the whole device for its own arena at start-up and
 * hands plug-ins nothing but their input and output buffers; a processing loop with a latency bound, where
 * cudaMalloc / cudaFree would stall every stream of the device; a process held to a device-memory quota that is
 * already spent.  sim_accumulate_static is steps A1-A7 (the same production accumulation kernel and the same
 * finalize kernel as sim_accumulate_update) for ONE update with no handle and no workspace: the
 * fp64 accumulator and the scheduling counters of the kernel live in a fixed array compiled into libsim.so
 * (SIM_STATIC_MAX_CELLS fp64 pairs = 1 MiB, plus 256 bytes of counters; every GPU on which the library is used holds
 * that much until the process exits).  The call itself allocates nothing: no cudaMalloc, no cudaFree, no library
 * routine that allocates.
 *
 *   cfg         HOST.  n_gates, n_doppler, wavelength_m, prf_hz, gate_spacing_m, antenna_alpha, doppler_mode and device
 *               are used; the other fields must merely be valid (see sim_config).  n_gates * n_doppler must not exceed
 *               SIM_STATIC_MAX_CELLS (all five BASELINE configs fit: 128 x 512 at most): SIM_ERR_BAD_CONFIG otherwise.
 *   d_scat      DEVICE arrays as for sim_accumulate_update (16-byte aligned; n may be 0).
 *   sat         HOST, read during the call.
 *   d_spectrum  DEVICE, complex64 [n_gates][n_doppler], bin fastest, 16-byte aligned, owned by the caller.
 *               flags = 0: overwritten with the update's spectrum.  flags = SIM_ACC_APPEND: the batch is added to what
 *               it holds (scenes delivered in pieces).
 *   cuda_stream a cudaStream_t on cfg->device (NULL = legacy default stream); the work is enqueued, not waited for.
 *
 * The analytic antenna gain only (a tabulated pattern belongs to a handle).
 * First call on a device: the library looks up the device address of its array and reads three device attributes
 * (once per device, kept for later calls), and the CUDA runtime loads the kernels.  Make that first call during
 * start-up, outside any stream capture.
 * The array is shared by every call in the process.  Each call clears the part it uses before the kernel runs, so
 * nothing is carried over from the call before; but two calls whose GPU work overlaps in time (different streams, or
 * different host threads on different streams) race on it and both results are garbage: keep all calls of a device
 * on one stream, or order them with events.  Calls on different devices do not interact.
 * Errors: SIM_ERR_INVALID_ARG (NULL / misaligned pointers, unknown flag), SIM_ERR_BAD_CONFIG (invalid cfg, too many
 * cells, gate window too deep), SIM_ERR_CUDA.  Message: sim_last_error(NULL) on the calling thread. */
#define SIM_STATIC_MAX_CELLS 65536
int sim_accumulate_static(const sim_config* cfg, const sim_scatterers* d_scat, const sim_sat_state* sat,
                          void* d_spectrum, void* cuda_stream, uint32_t flags);

/* Message of the last error on this handle ("" if none); valid until the next call.  h may be NULL
 * (returns the message of the last failed sim_create / sim_workspace_bytes on this thread). */
const char* sim_last_error(const sim_handle* h);

#ifdef __cplusplus
}
#endif
#endif /* PAPER_2408_11472_SIM_H */
