/*
 * bloch.h -- C ABI of libbloch_b200: the spin-parallel Bloch-equation solve of KomaMRI (arxiv 2301.02702)
 * as hand-written CUDA for sm_100a.
 *
 * The calls follow the paper's problem statement (Fig 3 :188): scanner parameters +
 * phantom + sequence (+ simulation parameters) in; raw complex signal per ADC sample, and optionally the
 * final magnetisation, out.  No torch types, no C++ types, no exceptions across this boundary.
 *
 * Conventions
 *   - SI units: position [m], gradient [T/m], B1 [T], off-resonance [rad/s], time [s], gamma [rad/s/T].
 *   - Every function returns 0 (BLOCH_OK) or a negative bloch_status; bloch_last_error() gives thread-local
 *     detail text.  Nothing is printed, nothing aborts.
 *   - "h_" pointers are HOST memory, "d_" pointers are DEVICE memory of the current CUDA device.
 *   - The library never allocates device memory: tables, workspace and all spin / signal buffers are
 *     caller-owned (in this repo: torch tensors).  Host arrays passed to bloch_plan_create are borrowed
 *     for the duration of that call only.
 *   - The library reads no environment variable: kernel selection is plan state (bloch_plan_set_option).
 *   - `stream` arguments are a cudaStream_t passed as void* (NULL = legacy default stream).
 *   - Complex values are interleaved (re, im) fp32 pairs.
 */
#ifndef BLOCH_B200_H
#define BLOCH_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    BLOCH_OK = 0,
    BLOCH_EINVAL = -1,         /* NULL pointer, negative size, non-finite value, bad enum */
    BLOCH_ENONMONOTONIC = -2,  /* gradient vertex / RF sample / ADC times not ascending, or RF samples overlap */
    BLOCH_EADC_IN_RF = -3,     /* (not returned any more: ADC samples inside an RF run are served, reading G7) */
    BLOCH_EWORKSPACE = -4,     /* workspace / table buffer too small or misaligned (256 B) */
    BLOCH_ECUDA = -5,          /* a CUDA runtime call failed; text in bloch_last_error() */
    BLOCH_EARCH = -6,          /* current device is not compute capability 10.x */
    BLOCH_ENOTUPLOADED = -7,   /* bloch_simulate before bloch_plan_upload */
    BLOCH_ENOMEM = -8,         /* host allocation failed */
    BLOCH_EHWLIMIT = -9,       /* a gradient vertex exceeds scanner G_max, or a segment exceeds S_max (when given) */
    BLOCH_ERANGE = -10         /* the phantom lies outside what the plan's phase mode resolves (see bloch_sim_params) */
} bloch_status;

enum { BLOCH_PHASE_AUTO = 0, BLOCH_PHASE_FP32 = 1, BLOCH_PHASE_FP64 = 2 };
enum { BLOCH_OUT_SUM_ALL = 0, BLOCH_OUT_PER_SPIN = 1, BLOCH_OUT_GROUPED = 2 };
enum { BLOCH_MOTION_NONE = 0, BLOCH_MOTION_LINEAR = 1, BLOCH_MOTION_WAVEFORM = 2 };

/* Scanner.  Only gamma enters the arithmetic (Eq 1-2, :105-114); B0, G_max, S_max are
 * limits: when G_max [T/m] or S_max [T/m/s] is > 0, bloch_plan_create checks every gradient vertex and every
 * segment between vertices against it, per axis, and returns BLOCH_EHWLIMIT; 0 = not checked.  B0 is carried
 * only.  gamma <= 0 selects 2*pi*42.58e6 (:322). */
typedef struct {
    double gamma;
    double B0;
    double G_max;
    double S_max;
} bloch_scanner;

/* Sequence: G(t) piecewise linear through per-axis vertices (G = 0 outside the vertex range,
 * :180), complex B1(t) piecewise constant on [rf_t, rf_t + rf_dt) (:182), ADC sample times.  All times in
 * [0, t_end], each array strictly ascending; RF samples may abut but not overlap. */
typedef struct {
    const double *g_t[3];
    const double *g_v[3];
    int64_t g_n[3];
    const double *rf_t;
    const double *rf_dt;
    const double *rf_re;
    const double *rf_im;
    int64_t rf_n;
    const double *adc_t;
    int64_t adc_n;
    double t_end;
} bloch_sequence;

/* simParams.  dt_rf_max: RF sample pieces longer than this are cut into equal sub-steps
 * (the paper's dt_rf, :182).  dt_max: with motion_mode != NONE every interval longer than this is cut into
 * equal sub-steps (the paper's "intermediate points in the case of motion", :180); ignored without motion
 * or when <= 0 / inf.  motion_mode: BLOCH_MOTION_LINEAR builds the first-moment tables that let every spin
 * move as x(t) = x + v t (PAPER.md:96 motion field, :236 experiment (d)); velocities are given to
 * bloch_simulate_motion.  BLOCH_MOTION_WAVEFORM is the general form x(t) = x + a u(t) ("motion field
 * u(x, t)"; reading M2): u is ONE piecewise-linear waveform shared by all spins, given here by its vertices
 * (motion_t strictly ascending [s], motion_u [any unit], motion_n >= 1; HOST arrays borrowed for the duration of
 * bloch_plan_create; u keeps its end values outside the vertices, and the vertices inside [0, t_end] join the time
 * grid), and a is the per-spin amplitude vector [m per unit of u] passed to bloch_simulate_motion in place of the
 * velocities -- periodic (cardiac, respiratory) displacement, stop-and-go, pulsatile flow; u(t) = t is MOTION_LINEAR.
 * The effective field is sampled at the interval ends and integrated by the paper's trapezoid on the dt_max-refined
 * grid either way, so one more spin-independent table (the moment of G u) serves every spin.
 * max_block_points: precession blocks hold at most
 * this many evaluated points (the paper's Nblocks memory bound, :171); <= 0 selects the default. */
typedef struct {
    double dt_max;
    double dt_rf_max;
    int64_t max_block_points;
    int32_t phase_mode;   /* BLOCH_PHASE_* */
    int32_t output_mode;  /* BLOCH_OUT_*   */
    int32_t motion_mode;  /* BLOCH_MOTION_* */
    int32_t group_size;   /* BLOCH_OUT_GROUPED: spins per group (>= 1; n_spins must be a multiple); else ignored */
    /* Extents of the phantoms this plan will be run on.  The plan is spin-independent (it is built from the sequence
     * alone), so what BLOCH_PHASE_AUTO needs to know about the spins is declared here: the fp32 phase of the signal
     * kernels resolves 2^-24 of the largest block-relative phase, bounded by |k| max_extent_m + max_offres_hz tau
     * (+ |first moment| max_speed_mps with motion), and AUTO takes fp64 phase accumulation above 256 turns.
     * <= 0 selects 0.25 m / 1000 Hz / 1 m/s.  Every bloch_simulate measures the phantom it is given (max |x|,
     * max |dw|, max |v|) and reports BLOCH_ERANGE through bloch_plan_status when an AUTO plan that resolved to fp32
     * would pass 256 turns with it, or an fp64-phase plan 2^19 turns (the limit of its fixed-point phase fraction);
     * a plan whose declared extents already pass 2^19 turns is rejected by bloch_plan_create (BLOCH_ERANGE).
     * A plan forced to BLOCH_PHASE_FP32 is not checked: the caller has taken the phase precision on. */
    double max_extent_m;   /* largest |x| (Euclidean norm) of any spin [m] */
    double max_offres_hz;  /* largest |dw| / 2 pi [Hz] */
    double max_speed_mps;  /* largest |v| [m/s] (MOTION_LINEAR) or amplitude |a| [m per unit of u] (MOTION_WAVEFORM) */
    const double *motion_t;  /* BLOCH_MOTION_WAVEFORM: vertex times of u(t), strictly ascending; else ignored */
    const double *motion_u;  /*                        vertex values */
    int64_t motion_n;
} bloch_sim_params;

typedef struct {
    int64_t n_intervals;     /* intervals of the merged, refined time grid (what a step-by-step solver runs) */
    int64_t n_rf_steps;      /* RF-active intervals */
    int64_t n_adc;           /* ADC samples */
    int64_t n_blocks;        /* excitation + precession blocks */
    int64_t n_rf_blocks;
    int64_t n_eval_points;   /* precession evaluations per spin: ADC samples + block ends */
    int64_t n_launches;      /* kernels one bloch_simulate enqueues for this plan (SUM_ALL, final state on) */
    int64_t table_bytes;     /* size of the device table buffer bloch_plan_upload needs */
    int64_t max_block_adc;   /* largest number of ADC samples in one precession block */
    int32_t phase_mode;      /* resolved: BLOCH_PHASE_FP32 or BLOCH_PHASE_FP64 */
    int32_t output_mode;
    int32_t motion_mode;
    int32_t group_size;
    int32_t phase_mode_requested;  /* as given: BLOCH_PHASE_AUTO / FP32 / FP64 */
    int32_t path;            /* BLOCH_PATH_* as set by bloch_plan_set_path */
    double max_extent_m;     /* the extents the plan assumes (bloch_sim_params, defaults resolved) */
    double max_offres_hz;
    double max_speed_mps;
    double worst_turns;      /* largest block-relative phase [turns] any evaluated point can reach within those extents */
    int32_t options[16];     /* current BLOCH_OPT_* values (bloch_plan_set_option) */
} bloch_plan_info;

typedef struct bloch_plan bloch_plan;

int bloch_version(void);
const char *bloch_strerror(int code);
const char *bloch_last_error(void);

/* Host only: merge the time grid, interpolate G, classify intervals into excitation
 * / precession blocks (:132, :171), precompute per precession block the spin-independent cumulative
 * gradient moment k(t) by the trapezoidal rule on the vertices (Eq 12-13, :173-180) and per RF step the
 * rotation-vector table.  *out is owned by the library until bloch_plan_destroy. */
int bloch_plan_create(const bloch_scanner *scanner, const bloch_sequence *seq,
                      const bloch_sim_params *params, bloch_plan **out);
int bloch_plan_destroy(bloch_plan *plan);
int bloch_plan_get_info(const bloch_plan *plan, bloch_plan_info *out);

/* The plan's table image in HOST memory: *h_tables points at table_bytes bytes owned by the plan (borrowed until it is
 * destroyed) -- what bloch_plan_upload copies to the device.  For callers that upload by other means, and for tests
 * that compare plans. */
int bloch_plan_host_tables(const bloch_plan *plan, const void **h_tables, size_t *bytes);

/* Bytes of caller-allocated device workspace bloch_simulate needs for n_spins (256-B aligned buffer). */
int bloch_plan_workspace_bytes(const bloch_plan *plan, int64_t n_spins, size_t *out);

/* Copy the plan's tables into d_tables (>= table_bytes, 256-B aligned, caller keeps it alive until the
 * plan is destroyed or re-uploaded).  Asynchronous on `stream`; the host staging copy is owned by the plan. */
int bloch_plan_upload(bloch_plan *plan, void *d_tables, size_t bytes, void *stream);

/* Run the whole sequence for n_spins spins (device pointers, fp32 SoA arrays of n_spins each).
 *   d_Mxy (2*n_spins floats, interleaved) / d_Mz: if init_equilibrium == 0 they hold the initial state
 *       (both required); if non-NULL they receive the final magnetisation.  With init_equilibrium != 0
 *       the state starts at Mxy = 0, Mz = M0 (reading G8).
 *   d_signal: SUM_ALL: n_adc complex, S[j] = sum over spins of Mxy at ADC sample j;
 *             PER_SPIN: n_spins x n_adc complex, row-major [spin][adc];
 *             GROUPED: (n_spins / group_size) x n_adc complex, row-major [group][adc],
 *             S[g][j] = sum of Mxy over the group_size consecutive spins of group g -- an isochromat ensemble
 *             per voxel or per dictionary entry.
 *   Asynchronous on `stream`: no hidden synchronisation, no allocation, no host copies.  The result is
 *   bitwise reproducible run to run (no floating-point atomics).  T1, T2 must be > 0 and finite: checked on the
 *   device by the first kernel, reported by bloch_plan_status / the next call (BLOCH_EINVAL).
 * The call only enqueues work on `stream` (kernels and memsets; CUDA events too when profiling is on): it may be
 * captured into a CUDA graph by the caller and replayed. */
int bloch_simulate(const bloch_plan *plan, int64_t n_spins,
                   const float *d_x, const float *d_y, const float *d_z, const float *d_M0,
                   const float *d_T1, const float *d_T2, const float *d_dw,
                   float *d_Mxy, float *d_Mz, int init_equilibrium,
                   float *d_signal, void *d_workspace, size_t workspace_bytes, void *stream);

/* bloch_simulate for a moving phantom: spin i is at x_i + v_i t at sequence time t.
 * d_vx, d_vy, d_vz: fp32 device arrays [m/s] of n_spins each; the plan must have been created with
 * motion_mode = BLOCH_MOTION_LINEAR or BLOCH_MOTION_WAVEFORM (else BLOCH_EINVAL); with a waveform plan they hold the
 * amplitude vectors a_i of x_i(t) = x_i + a_i u(t) [m per unit of u].  All three NULL = bloch_simulate.  The effective
 * field is sampled at the ends of every interval of the dt_max-refined grid and integrated by the trapezoidal
 * rule exactly as the paper prescribes (:180, :336); because x(t) is linear in t this needs only one more
 * spin-independent table, the first moment sum of (G_n t_n + G_{n+1} t_{n+1}) dt_n / 2. */
int bloch_simulate_motion(const bloch_plan *plan, int64_t n_spins,
                          const float *d_x, const float *d_y, const float *d_z, const float *d_M0,
                          const float *d_T1, const float *d_T2, const float *d_dw,
                          const float *d_vx, const float *d_vy, const float *d_vz,
                          float *d_Mxy, float *d_Mz, int init_equilibrium,
                          float *d_signal, void *d_workspace, size_t workspace_bytes, void *stream);

/* Same computation with HOST buffers (pageable or pinned): copies the seven phantom arrays (and the initial
 * state, if any) to the device, runs bloch_simulate, copies the signal (and final state, if requested)
 * back and synchronises `stream` before returning.  d_scratch is caller-allocated device memory of at
 * least bloch_simulate_host_scratch_bytes(); the tables must have been uploaded. */
int bloch_simulate_host_scratch_bytes(const bloch_plan *plan, int64_t n_spins, size_t *out);
int bloch_simulate_host(const bloch_plan *plan, int64_t n_spins,
                        const float *h_x, const float *h_y, const float *h_z, const float *h_M0,
                        const float *h_T1, const float *h_T2, const float *h_dw,
                        float *h_Mxy, float *h_Mz, int init_equilibrium,
                        float *h_signal, void *d_scratch, size_t scratch_bytes, void *stream);

/* Host-buffer variant of bloch_simulate_motion (h_vx, h_vy, h_vz host arrays, all three NULL = no motion);
 * scratch as bloch_simulate_host_scratch_bytes. */
int bloch_simulate_host_motion(const bloch_plan *plan, int64_t n_spins,
                               const float *h_x, const float *h_y, const float *h_z, const float *h_M0,
                               const float *h_T1, const float *h_T2, const float *h_dw,
                               const float *h_vx, const float *h_vy, const float *h_vz,
                               float *h_Mxy, float *h_Mz, int init_equilibrium,
                               float *h_signal, void *d_scratch, size_t scratch_bytes, void *stream);

/* bloch_simulate for callers that cannot allocate device memory (code under CUDA graph capture, tight serving loops,
 * harnesses that forbid cudaMalloc): the same computation for a static plan (BLOCH_MOTION_NONE; any output mode, phase
 * mode and path), but the workspace -- the packed spin records and the per-chunk partial signal rows of the two-pass
 * reduction -- is a device array of BLOCH_STATIC_WORKSPACE_BYTES inside
 * the library, which every GPU context that loads the library holds until it exits.  The caller passes only inputs
 * and outputs (device pointers, as bloch_simulate); the tables must have been uploaded into caller memory.
 *   - Allocates nothing: no cudaMalloc / cudaFree / cudaHostAlloc / event or stream creation, on any path.  Plans with
 *     profiling switched on are refused (BLOCH_EINVAL: the taps create CUDA events), motion plans too.
 *   - BLOCH_EWORKSPACE (text in bloch_last_error) when bloch_plan_workspace_bytes(plan, n_spins) exceeds
 *     BLOCH_STATIC_WORKSPACE_BYTES: nothing is enqueued; use bloch_simulate with a caller workspace.  Sizes that fit:
 *     e.g. the whole of config 3 (131,072 spins, fp64 phase: 20.2 MB), config 2 (1.3 MB), config 5 (12.8 MB) and
 *     config 5b (4.8 MB); ~595,000 spins of an fp32-phase plan with short blocks (config 4's 1,000,000 need 203 MB).
 *   - Every call on a device shares the ONE array, which keeps the previous call's contents; the call clears what must
 *     start at zero on `stream` itself.  Two calls whose GPU work overlaps (different streams, or one stream per
 *     thread) RACE on the array: serialise them (one stream, or an event between them).  Results are bitwise those of
 *     bloch_simulate.  Asynchronous on `stream`, no synchronisation. */
#define BLOCH_STATIC_WORKSPACE_BYTES (32u << 20)
int bloch_simulate_static(const bloch_plan *plan, int64_t n_spins,
                          const float *d_x, const float *d_y, const float *d_z, const float *d_M0,
                          const float *d_T1, const float *d_T2, const float *d_dw,
                          float *d_Mxy, float *d_Mz, int init_equilibrium,
                          float *d_signal, void *stream);

/* Timing taps for the benchmark.  With bloch_plan_set_profiling(plan, 1) bloch_simulate records one CUDA
 * event on `stream` before every kernel it launches (and one after the last); off by default.  After the
 * caller has synchronised `stream`, bloch_plan_last_timing fills, per kernel kind, the summed device time
 * [ms] and the number of launches of the last bloch_simulate: arrays of BLOCH_N_KINDS entries indexed by
 * BLOCH_KIND_*.  A kernel's time is the interval to the next event on the stream, so it includes the
 * launch gap that follows it. */
enum { BLOCH_KIND_OTHER = 0,   /* pack / unpack / block-end propagation only */
       BLOCH_KIND_RF = 1,      /* excitation kernel */
       BLOCH_KIND_SIGNAL = 2,  /* free-precession signal kernel (a6) */
       BLOCH_KIND_REDUCE = 3,  /* second pass of the signal reduction (a7) */
       BLOCH_KIND_FUSED = 4,   /* whole-sequence kernel (a5-a8 in one launch, BLOCH_PATH_FUSED) */
       BLOCH_N_KINDS = 5 };
int bloch_plan_set_profiling(bloch_plan *plan, int enable);
int bloch_plan_last_timing(const bloch_plan *plan, float *ms_by_kind, int64_t *launches_by_kind);
/* Number of kernels the last bloch_simulate on this plan enqueued (it depends on n_spins through the batching
 * of the second-pass reduction; bloch_plan_info.n_launches is the upper bound with one second pass per block). */
int bloch_plan_last_launches(const bloch_plan *plan, int64_t *out);
/* The largest launch (threads in flight) of kernel kind `kind` in the last bloch_simulate on this plan: its name as a
 * profiler prints it (e.g. "rf_kernel<0>", "signal_kernel<8, 0, 0>"; empty if the kind did not run), CTAs in the
 * grid and threads per CTA.  The benchmark uses it to decide whether a committed ncu capture describes the kernel
 * it has just timed.  name: caller's buffer of name_bytes (may be NULL); grid_ctas, block_threads may be NULL. */
int bloch_plan_last_kernel(const bloch_plan *plan, int kind, char *name, size_t name_bytes, int64_t *grid_ctas,
                           int *block_threads);

/* Multi-coil receive (SURVEY.md 8(f) f2 "per-coil weights"; PAPER.md:95 "coil sensitivity", :372; reading C1 of
 * DESIGN.md): S_c(t_n) = sum_i C_c(x_i) Mxy_i(t_n) for n_coils receive coils.
 *   d_coil    DEVICE, float2 [n_coils][n_spins] row-major: complex sensitivity of coil c at spin i (re, im); borrowed
 *   d_signal  DEVICE, float2 [n_coils][n_adc] row-major, written
 *   workspace as bloch_simulate, sized by bloch_plan_workspace_bytes_coils(plan, n_spins, n_coils)
 * Everything else as bloch_simulate (same integration, same final magnetisation).  The plan must be BLOCH_OUT_SUM_ALL
 * (else BLOCH_EINVAL); 1 <= n_coils <= 4096.  Moving spins: bloch_simulate_coils_motion (motion plans; velocities /
 * amplitudes as bloch_simulate_motion, all three NULL = none).  The coil-independent part of every evaluation (phase,
 * sin / cos / exp) is computed once per pass of coils; with fp32 phase and static spins the sum over spins runs on the
 * tensor cores (tcgen05 with the generated operand in tensor memory, two FP16 pieces per value with FP32 accumulation
 * -- 22 significant bits, as 3xTF32 --, 8, 16 or 32 coils per pass).  Plans that
 * take the whole-sequence kernel (BLOCH_PATH_FUSED, or AUTO where it qualifies: static spins, fp32 phase) sum up to 8
 * coils inside that one launch; more coils, or 8 coils on blocks large enough for the tensor-core kernel, run block by
 * block (BLOCH_PATH_FUSED with more than 8 coils: BLOCH_EINVAL).  Asynchronous on `stream`; never allocates. */
int bloch_plan_workspace_bytes_coils(const bloch_plan *plan, int64_t n_spins, int n_coils, size_t *out);
int bloch_simulate_coils(const bloch_plan *plan, int64_t n_spins, const float *d_x, const float *d_y,
                         const float *d_z, const float *d_M0, const float *d_T1, const float *d_T2,
                         const float *d_dw, int n_coils, const float *d_coil, float *d_Mxy, float *d_Mz,
                         int init_equilibrium, float *d_signal, void *d_workspace, size_t workspace_bytes,
                         void *stream);

int bloch_simulate_coils_motion(const bloch_plan *plan, int64_t n_spins, const float *d_x, const float *d_y,
                                const float *d_z, const float *d_M0, const float *d_T1, const float *d_T2,
                                const float *d_dw, const float *d_vx, const float *d_vy, const float *d_vz, int n_coils,
                                const float *d_coil, float *d_Mxy, float *d_Mz, int init_equilibrium, float *d_signal,
                                void *d_workspace, size_t workspace_bytes, void *stream);

/* Host-buffer variant of bloch_simulate_coils: phantom, coil weights (float2 [n_coils][n_spins]), state and signal
 * (float2 [n_coils][n_adc]) are HOST arrays (pinned memory makes the copies asynchronous); H2D and D2H copies are
 * made on `stream` inside the call, which synchronises the stream before returning.  d_scratch: DEVICE, 256-B
 * aligned, at least bloch_simulate_host_coils_scratch_bytes(). */
int bloch_simulate_host_coils_scratch_bytes(const bloch_plan *plan, int64_t n_spins, int n_coils, size_t *out);
int bloch_simulate_host_coils(const bloch_plan *plan, int64_t n_spins, const float *h_x, const float *h_y,
                              const float *h_z, const float *h_M0, const float *h_T1, const float *h_T2,
                              const float *h_dw, int n_coils, const float *h_coil, float *h_Mxy, float *h_Mz,
                              int init_equilibrium, float *h_signal, void *d_scratch, size_t scratch_bytes,
                              void *stream);
int bloch_simulate_host_coils_motion(const bloch_plan *plan, int64_t n_spins, const float *h_x, const float *h_y,
                                     const float *h_z, const float *h_M0, const float *h_T1, const float *h_T2,
                                     const float *h_dw, const float *h_vx, const float *h_vy, const float *h_vz,
                                     int n_coils, const float *h_coil, float *h_Mxy, float *h_Mz, int init_equilibrium,
                                     float *h_signal, void *d_scratch, size_t scratch_bytes, void *stream);

/* Execution path of bloch_simulate for this plan.
 *   BLOCH_PATH_PER_BLOCK: one excitation launch per RF block and one signal launch per precession block.
 *   BLOCH_PATH_FUSED: ONE persistent whole-sequence launch (a CTA per SM owns a chunk of spins for the whole
 *       sequence; warp-specialised excitation / readout, see csrc/seq.cuh) plus the second-pass reduction.
 *       Available for SUM_ALL output (and for PER_SPIN plans whose blocks hold at most 16 ADC samples: dictionary
 *       mode), fp32 phase, no motion and at most 29 x 32 spins per SM; bloch_simulate
 *       returns BLOCH_EINVAL when it is forced and not available.
 *   BLOCH_PATH_AUTO (default): FUSED when available, 4 N_rf >= N_adc and the signal warps of the balanced layout fit
 *       beside the RF warps (up to about 20 x 32 spins per SM), else PER_BLOCK.
 * Both paths compute the same thing; the final magnetisation is bitwise identical, the signal differs only in
 * the order of the fixed-order sums.  Set before bloch_plan_workspace_bytes: the workspace size depends on it. */
enum { BLOCH_PATH_AUTO = 0, BLOCH_PATH_PER_BLOCK = 1, BLOCH_PATH_FUSED = 2 };
int bloch_plan_set_path(bloch_plan *plan, int path);

/* Kernel-selection options of a plan: which of the library's kernels / launch shapes bloch_simulate takes where it has
 * a choice.  They are state of the PLAN (set once, echoed in bloch_plan_info.options), never ambient process state:
 * the library reads no environment variable.  Defaults are what DESIGN.md's measurements use; every setting computes
 * the same thing (tests compare them against each other and against the oracle).  Set before
 * bloch_plan_workspace_bytes: launch shapes enter the workspace size.  Unknown key or value out of range: BLOCH_EINVAL.
 *   BLOCH_OPT_SIGNAL_LIN          1 (default): Cartesian readouts (k' advances by a constant step) take the rotation
 *                                 recurrence; 0: every sample takes its own sin / cos
 *   BLOCH_OPT_SIGNAL_P            0 (default): the library picks 1, 2, 4 or 8 adjacent ADC samples per thread of the
 *                                 signal kernel from the block length; 1 / 2 / 4 / 8 forces it
 *   BLOCH_OPT_SIGNAL_FIXED_CTA    0 (default): readouts of fewer than 256 samples get CTAs of just enough warps; 1: 256
 *   BLOCH_OPT_SIGNAL_CTAS_PER_SM  resident signal CTAs per SM the grid is sized for: 1..8, default 4
 *   BLOCH_OPT_RF_THREADS          0 (default): 128-thread excitation CTAs once there are >= 32 warps per SM, else 32;
 *                                 32 / 64 / 128 forces it
 *   BLOCH_OPT_RF_SPINS            spins per thread of the excitation kernel: 0 (default) the library's choice, 1 or 2
 *   BLOCH_OPT_COIL_TC             multi-coil receive: tensor cores (tcgen05, A operand in tensor memory) whenever
 *                                 they apply (fp32 phase, static spins): -1 (default) and 2 with FP16 operand
 *                                 pieces scaled from measured maxima (2 instructions per 8 spins; any number of coils
 *                                 from 4096 spins on), 1 with 3xTF32 (4 instructions; more than 4 coils); 0: never
 *                                 (the FFMA kernel)
 *   BLOCH_OPT_SEQ_SIG_EXTRA       whole-sequence kernel: signal warps added per missing RF warp of a sub-partition,
 *                                 0..7; -1 (default): 2, or 0 with receive coils
 *   BLOCH_OPT_SEQ_SIG_BASE        whole-sequence kernel: signal warps per sub-partition, 0..7; -1 (default) automatic
 *   BLOCH_OPT_SEQ_ITEMS_X4        whole-sequence kernel: readout items per signal warp x 4 that the item size must
 *                                 leave; 0 (default) always the largest item
 *   BLOCH_OPT_RF_CONST            1 (default): from 16,384 spins on, excitation blocks of static plans whose gradient
 *                                 is constant within every tile take rf_const_kernel -- the step records passed by
 *                                 value as kernel parameters (constant bank, uniform operands; blocks of up to 2000
 *                                 steps in up to 24 tiles, longer ones keep the tile kernel); 2: for any number of
 *                                 spins; 0: always the shared-memory tile kernel.  Bitwise the same result. */
enum { BLOCH_OPT_SIGNAL_LIN = 0, BLOCH_OPT_SIGNAL_P = 1, BLOCH_OPT_SIGNAL_FIXED_CTA = 2,
       BLOCH_OPT_SIGNAL_CTAS_PER_SM = 3, BLOCH_OPT_RF_THREADS = 4, BLOCH_OPT_RF_SPINS = 5, BLOCH_OPT_COIL_TC = 6,
       BLOCH_OPT_SEQ_SIG_EXTRA = 7, BLOCH_OPT_SEQ_SIG_BASE = 8, BLOCH_OPT_SEQ_ITEMS_X4 = 9, BLOCH_OPT_RF_CONST = 10,
       BLOCH_N_OPTIONS = 11 };
int bloch_plan_set_option(bloch_plan *plan, int key, int value);
int bloch_plan_get_option(const bloch_plan *plan, int key, int *value);

/* What the last bloch_simulate* on this plan found out about the phantom it was given.  pack_kernel (the first
 * kernel of every simulation) checks every spin -- T1, T2 > 0 and finite (they enter as 1/T1, 1/T2),
 * every value finite -- and measures max |x|, max |dw|, max |v|; the findings (32 bytes) follow the simulation on
 * `stream` into pinned host memory owned by the plan (allocated by bloch_plan_upload, so bloch_simulate still never
 * allocates and never synchronises).
 *   bloch_plan_status synchronises `stream`, evaluates them, clears them, stores the BLOCH_STATUS_* bits in *flags
 *   (may be NULL) and returns BLOCH_OK, BLOCH_EINVAL (bad T1 / T2 / non-finite input) or BLOCH_ERANGE (phase range,
 *   see bloch_sim_params).  The host-buffer entries (bloch_simulate_host*) make this check themselves before they
 *   return.  A device-buffer bloch_simulate* whose predecessor on the same plan left findings that nobody collected
 *   returns that error instead of running ("fails on the next call"), and clears them. */
enum { BLOCH_STATUS_BAD_RELAXATION = 1, BLOCH_STATUS_NONFINITE = 2, BLOCH_STATUS_PHASE_RANGE = 4 };
int bloch_plan_status(const bloch_plan *plan, void *stream, int *flags);
/* *out = 1 if bloch_simulate would take the fused path for n_spins on the current device, else 0. */
int bloch_plan_uses_fused(const bloch_plan *plan, int64_t n_spins, int *out);

/* Files (PAPER.md:93 Fig 1 "each arrow represents a file", :99-101).  The paper reads Pulseq sequence files and writes
 * ISMRM Raw Data but fixes nothing of either format, and neither can be checked against anything here; these calls read
 * and write THIS LIBRARY'S OWN line-oriented text container for exactly the arrays of bloch_scanner / bloch_sequence and
 * for the raw samples (layout: csrc/io.cpp) -- not Pulseq, not ISMRMRD.  Numbers are C99 hexadecimal floating-point
 * literals, so a round trip is bit-exact: a plan built from a file has bitwise the tables of a plan built from the
 * arrays.  Host only; all pointers are HOST memory.
 *   bloch_sequence_write      scanner may be NULL (zeros are written).
 *   bloch_sequence_read       *out is owned by the library until bloch_sequence_file_free.
 *   bloch_sequence_file_get   fills *scanner (may be NULL) and *seq with pointers INTO the file object (borrowed; valid
 *                             until it is freed), ready for bloch_plan_create.
 *   bloch_signal_write        h_signal: n_rows x n_adc interleaved (re, im) fp32 (rows = 1, coils, spins or groups);
 *                             h_adc_t (n_adc sample times) may be NULL.
 *   bloch_signal_read         with h_signal == NULL only *n_rows and *n_adc are returned; else capacity_complex >=
 *                             n_rows x n_adc (BLOCH_EWORKSPACE otherwise); h_adc_t may be NULL.
 * Errors: BLOCH_EINVAL (cannot open, malformed, wrong magic), BLOCH_ENOMEM. */
typedef struct bloch_sequence_file bloch_sequence_file;
int bloch_sequence_write(const char *path, const bloch_scanner *scanner, const bloch_sequence *seq);
int bloch_sequence_read(const char *path, bloch_sequence_file **out);
int bloch_sequence_file_get(const bloch_sequence_file *file, bloch_scanner *scanner, bloch_sequence *seq);
int bloch_sequence_file_free(bloch_sequence_file *file);
int bloch_signal_write(const char *path, const float *h_signal, int64_t n_rows, int64_t n_adc, const double *h_adc_t);
int bloch_signal_read(const char *path, float *h_signal, int64_t capacity_complex, int64_t *n_rows, int64_t *n_adc,
                      double *h_adc_t);

/* Pipe micro-benchmarks used for the roofline denominators (MEASURED_PEAKS.json has only HBM and bf16):
 * kind 0 = MUFU (sin/cos/ex2 mix), 1 = FFMA (two operands reused), 2 = DFMA, 3 = FFMA with three different changing
 * register operands (register-file operand bandwidth, the bound of the RF step's cross products).  Runs `iters` dependent-chain iterations with 8
 * independent chains per thread on all SMs at full occupancy and returns operations per second. */
int bloch_microbench(int kind, int iters, double *ops_per_s, void *stream);

#ifdef __cplusplus
}
#endif
#endif /* BLOCH_B200_H */
