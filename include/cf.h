/* cf.h -- C ABI of libcf.so: the batched quadrotor simulation step of Crazyflow
 * (arxiv/paper_2606_01478) as hand-written sm_100a CUDA kernels.
 *
 * The calls follow the paper's problem statement: a simulator object holding M_worlds x N_drones drones
 * (PAPER.md:L23, L264), a control-interface level, stepping n steps at once (the XLA scan of
 * PAPER.md:L264 becomes one kernel launch with the state held in registers), and resets.
 * BASELINE.json:north_star names the four mandatory calls: cf_create, cf_reset, cf_step, cf_get_state.
 *
 * GENERAL RULES
 *  - Every function returns CF_OK (0) or a negative cf_status; none throws, aborts or prints.  cf_last_error()
 *    returns a thread-local description of the last failure.
 *  - Ownership: the CALLER owns every device byte (workspace, commands, records, outputs).  The library owns only
 *    the host handle and never allocates device memory (one exception to "only the host handle": cf_rollout_host
 *    creates a second stream and up to 16 events on first use, see there and cf_set_copy_stream).  Pointers named *_dev are device pointers, *_host are host
 *    pointers (pinned memory makes the copies asynchronous to the host but the *_host calls still synchronise the
 *    stream before returning).
 *  - Asynchrony: all *_dev calls enqueue on the bound CUDA stream (cf_set_stream, default stream 0) and return; there
 *    is no implicit synchronisation.  Launch errors are caught with cudaGetLastError -> CF_E_CUDA.
 *  - There is no CPU path: an unsupported combination returns CF_E_UNSUPPORTED.
 *
 * LAYOUTS (float32, component-major "planes"; i = w*N + n is the flat drone index, MN = M*N)
 *   state  [D][MN]     D = 17 first-principles: p(0-2) q(3-6; x y z w, scalar-last)
 *                                                               v(7-9) omega_body(10-12) Omega(13-16, rpm)
 *                      D = 13 abstracted:       p(0-2) Psi(3-5 roll pitch yaw) v(6-8) dPsi(9-11) f_Sigma(12)
 *   record [n_rec][D][MN]
 *   cmds   [K][MN] of float4 (CF_CMD_BUFFER) or [K] of float4 (CF_CMD_NOMINAL_PLUS_NOISE), 16-byte aligned:
 *            attitude (roll, pitch, yaw [rad], collective thrust [N]);  position (x, y, z [m], yaw [rad]);
 *            rotor (4 x rpm);  torque (tau_x, tau_y, tau_z [N m], collective thrust [N])
 *   ctrl   [14][MN]    i_R(0-2) i_p(3-5) held attitude cmd(6-9) held rotor cmd(10-13)
 *   wparam [P][M]      P = 14 FP: m Jx Jy Jz kf0 kf1 kf2 km0 km1 km2 cv_up cv_dn cd_up cd_dn;  P = 11 AB: m a[3] b[3] c[3] c_tau
 *
 * STEP SEMANTICS.  The simulator keeps a global step counter s
 * (uint32, 0 after reset).  For each of the n_steps physics steps of length 1/f_phys:
 *   (1) if (s - s0) % cmd_hold == 0 the command with index (s - s0)/cmd_hold is fetched (or formed from
 *       nominal + Philox noise);  (2) position-controller tick if s % (f_phys/f_pos) == 0;  (3) attitude-controller
 *       tick + motor mixer if s % (f_phys/f_att) == 0 (first-principles model);  (4) disturbance draw for this s;
 *   (5) explicit Euler or classical RK4 step with the inputs held, then quaternion renormalisation;  (6) s += 1;
 *   (7) obstacle minima updated with the new position;  (8) if record_every > 0 and s % record_every == 0 the state
 *       is written to record slot  s/record_every - s0/record_every - 1.
 * Controller ticks, record slots and Philox counters depend only on the global s, so one fused call and any split
 * into shorter calls (down to n_steps = 1, the interactive mode) give the same trajectory.
 */
#ifndef CF_H
#define CF_H
#include <stddef.h>
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef struct cf_sim cf_sim;   /* opaque host handle */

typedef enum {
  CF_OK = 0,
  CF_E_ARG = -1,          /* NULL / out-of-range argument */
  CF_E_SHAPE = -2,        /* sizes inconsistent (M*N >= 2^31, too few commands, non-integer rate ratio) */
  CF_E_STATE = -3,        /* cf_step / cf_set_state before the first cf_reset */
  CF_E_BUFFER = -4,       /* caller buffer too small or misaligned */
  CF_E_CUDA = -5,         /* CUDA runtime error (text in cf_last_error) */
  CF_E_UNSUPPORTED = -6   /* combination not built (e.g. rotor interface with the abstracted model) */
} cf_status;

enum { CF_MODEL_FIRST_PRINCIPLES = 0, CF_MODEL_ABSTRACTED = 1 };          /* PAPER.md:L296 / L334 */
enum { CF_EULER = 0, CF_RK4 = 1 };                                        /* BASELINE.json:configs */
enum { CF_IF_ROTOR = 0, CF_IF_TORQUE = 1, CF_IF_ATTITUDE = 2, CF_IF_POSITION = 3 };
enum { CF_CMD_BUFFER = 0, CF_CMD_NOMINAL_PLUS_NOISE = 1 };
enum { CF_AUX_COUNTERS = 0,      /* uint32[4]: s, attitude ticks, position ticks, records written */
       CF_AUX_MIN_DIST = 1,      /* float[M]: min over steps, drones of the world and obstacles of |p - c_j| - r_j */
       CF_AUX_CTRL = 2,          /* float[14][MN] */
       CF_AUX_WORLD_PARAMS = 3,  /* float[P][M] */
       CF_AUX_REC_TABLE = 4,     /* uint32[CF_REC_TABLE_CAP]: record slot (since reset) -> step counter */
       CF_AUX_MIN_D2 = 5,        /* float[8][MN]: running minimum squared centre distance per obstacle */
       CF_AUX_COST = 6,          /* float[MN]: rollout cost J (R27): running + terminal + clearance + collision */
       CF_AUX_EPS = 7,           /* float[4][MN]: AR(1) noise state; NaN = nothing drawn since the last re-arm
                                    (kept only when noise_beta != 0) */
       CF_AUX_COST_RUN = 8,      /* float[MN]: running part of the cost only */
       CF_AUX_NONFINITE = 9 };   /* uint32[2]: number of drones whose state holds a NaN / Inf, index of the first one
                                    (0xFFFFFFFF if none) -- a debug read-out computed on demand by its own small kernel,
                                    nothing is added to the rollout kernels */
#define CF_REC_TABLE_CAP 4096
#define CF_MAX_OBSTACLES 8

/* POD parameter block.  cf_default_params() fills the values of BASELINE.json:configs[0] / configs[2] and the
 * readings of DESIGN.md (limits, controller gains).  struct_size must equal sizeof(cf_params). */
typedef struct cf_params {
  uint32_t struct_size;
  int32_t  integrator, iface, cmd_source;
  int32_t  ab_thrust_dyn;            /* 1: Eq. (9) thrust lag; 0: f_Sigma == f_cmd (simplified model) */
  int32_t  init_mode;                /* 0 fixed (p = p0_lo, level), 1 uniform box + random axis-angle tilt, 2 grid */
  int32_t  grid_dims[3];
  int32_t  n_obstacles;              /* 0..8; > 0 switches the running minimum distance on */
  int64_t  world_offset;             /* global index of local world 0: Philox is keyed by the global world index,
                                        so a shard of worlds reproduces the same slice of the full run */
  float f_phys, f_att, f_pos;        /* Hz; f_phys/f_att and f_phys/f_pos must be integers >= 1 */
  /* plant, nominal (Eqs. (1)-(6)); rotor speeds in rpm */
  float mass, J[3], arm, kf[3], km[3] /* c0 + c1 W + c2 W^2 */, g;
  float cv_up, cv_dn, cd_up, cd_dn;  /* Eq. (6): accelerate / decelerate coefficients */
  float Jp, Ca[3];                   /* Eq. (5) rotor inertia, body drag; 0 = off */
  /* abstracted model, Eqs. (7)-(10) */
  float ab_a[3], ab_b[3], ab_c[3], ab_ctau, ab_cf;
  /* limits */
  float rpm_min, rpm_max, thrust_min, thrust_max, tilt_max;
  /* attitude controller (C5) and position controller (C7) */
  float kR[3], kW[3], kI[3], iR_max;
  float kp[3], kd[3], ki[3], ip_max[3];
  /* per-world multiplicative randomisation U[lo,hi] per slot (lo = hi = 1: off).
   * FP slots: 0 m, 1-3 J, 4 k_f, 5 k_m, 6 motor time constant.  AB slots: 0 m, 1-3 a, 4-6 b, 8-10 c, 11 c_tau. */
  float rnd_lo[12], rnd_hi[12];
  float dist_sigma;                  /* per-step Gaussian force disturbance [N], world frame; 0 = off */
  /* reset */
  float p0_lo[3], p0_hi[3], tilt0_max;
  float grid_spacing, grid_jitter, grid_origin[3];
  /* planning rollouts (config 3) */
  float obstacles[CF_MAX_OBSTACLES][4];   /* cx cy cz r */
  float noise_sigma[4], cmd_lo[4], cmd_hi[4];
  /* sampling-based planning (readings R25-R27), CF_CMD_NOMINAL_PLUS_NOISE only */
  float noise_beta;                  /* R25: AR(1) coefficient of the temporally correlated command noise in [0,1):
                                        eps <- z for the first command after a reset / cf_set_state, afterwards
                                        eps <- beta eps + sqrt(1 - beta^2) z;  command = clip(nominal + sigma eps) */
  int32_t n_ctrl;                    /* R26: number of nominal sequences (independent controllers), >= 1;
                                        the command buffer of cf_step is then [n_ctrl][n_cmds] float4 */
  int64_t worlds_per_ctrl;           /* controller of a world = LOCAL world index / worlds_per_ctrl (0: controller 0): the
                                        buffer holds this shard's controllers; the noise is keyed by the global world */
  int32_t cost_on;                   /* R27: accumulate the rollout cost (needs N == 1) */
  float cost_goal[3];                /* running cost per step: h (w_pos |p - goal|^2 + w_vel |v|^2), post-step state */
  float cost_w_pos, cost_w_vel;
  float cost_w_term;                 /* read-out adds w_term |p - goal|^2 of the current position, */
  float cost_w_obs, cost_d_safe;     /*   w_obs max(0, d_safe - d_min)^2 with d_min = CF_AUX_MIN_DIST of the drone, */
  float cost_w_coll;                 /*   and w_coll if d_min < 0 */
} cf_params;

/* Fill *p with the defaults for `model`.  Host only. */
void cf_default_params(cf_params *p, int model);
int  cf_state_dim(int model);          /* 17 / 13 */
int  cf_world_param_dim(int model);    /* 14 / 11 */

/* Bytes of device workspace cf_create needs for (M, N, model, p).  0 on invalid arguments. */
size_t cf_workspace_bytes(int64_t M, int64_t N, int model, const cf_params *p);

/* Create a simulator of M worlds x N drones.  workspace_dev: device memory of >= cf_workspace_bytes() bytes, 256-byte
 * aligned, owned by the caller and kept alive until cf_destroy.  Validates p (CF_E_ARG / CF_E_SHAPE /
 * CF_E_UNSUPPORTED), never touches the device. */
/* (Measurement switch: with CF_FORCE_GENERAL=1 in the environment at cf_create, cf_step always dispatches the general
 * run-time-gated kernel, also where a lean compile-time-selected one exists; results agree to rounding.) */
int cf_create(cf_sim **out, int64_t M, int64_t N, int model, const cf_params *p,
              void *workspace_dev, size_t workspace_bytes);
int cf_destroy(cf_sim *sim);

/* Bind the CUDA stream (a cudaStream_t, e.g. torch.cuda.current_stream().cuda_stream) all later calls enqueue on. */
int cf_set_stream(cf_sim *sim, void *cuda_stream);
/* The second stream cf_rollout_host queues its device->host result copies on.  By default the handle creates one of its
 * own on the first cf_rollout_host call; a caller that wants to own it (to give it a priority, or to order other work
 * against the copies) passes its stream here.  NULL returns to the library-owned stream.  The caller's stream must
 * outlive the handle or be replaced before it is destroyed; it must differ from the cf_set_stream stream for the copies
 * to overlap the next slice's kernel. */
int cf_set_copy_stream(cf_sim *sim, void *cuda_stream);

/* Draw the per-world parameters (Philox PARAM stream) and the initial state (INIT stream) from `seed`, zero the
 * controller integrals, set the held commands to hover, re-arm the minimum distance, s = 0.  (C9) */
int cf_reset(cf_sim *sim, uint64_t seed);

/* Continuous environment resets ("trivially handle continuous environment resets"): the worlds with
 * mask_dev[w] != 0 (uint8 [M], device) start a new episode -- initial state re-drawn from the INIT stream keyed by
 * episode_seed (same distributions as cf_reset), controller integrals 0, held commands = hover, minimum distance, noise
 * chain and rollout cost re-armed -- while every other world, the per-world parameters, the step counter and the seed of
 * the disturbance / noise streams stay untouched.  Needs a prior cf_reset. */
int cf_reset_masked(cf_sim *sim, const uint8_t *mask_dev, uint64_t episode_seed);

/* Overwrite the drone states: state_dev is [D][MN], or [D] broadcast to every drone when broadcast != 0 (the MPPI
 * "all rollouts start from the measured state" reset).  Keeps s and the world parameters; zeroes the
 * controller integrals, re-arms the minimum distance, held commands = hover.  Needs a prior cf_reset. */
int cf_set_state(cf_sim *sim, const float *state_dev, int broadcast);

/* Teacher forcing / checkpoint restore: overwrite any of state [D][MN], ctrl [14][MN], wparam [P][M],
 * min_d2 [8][MN] (NULL = keep) and, if step_counter >= 0, the global step counter. */
int cf_set_full(cf_sim *sim, const float *state_dev, const float *ctrl_dev, const float *wparam_dev,
                const float *min_d2_dev, int64_t step_counter);

/* Checkpoint restore of the counters cf_set_full leaves alone.  counters_host: the four words of CF_AUX_COUNTERS (step
 * counter s, attitude ticks, position ticks, records written) on the HOST; rec_table_dev: CF_REC_TABLE_CAP words as read
 * with CF_AUX_REC_TABLE, on the device, or NULL to keep the table.  Also sets the host mirror of s (cf_step_counter).
 * A COMPLETE CHECKPOINT of a simulator is: the seed given to cf_reset, cf_get_state, CF_AUX_CTRL, CF_AUX_WORLD_PARAMS,
 * CF_AUX_MIN_D2 (with obstacles), CF_AUX_EPS / CF_AUX_COST_RUN (planning rollouts), CF_AUX_COUNTERS, CF_AUX_REC_TABLE.
 * RESTORE into a simulator created with the same (M, N, model, params): cf_reset(seed); cf_set_full(state, ctrl, wparam,
 * min_d2, -1); cf_set_plan_state(eps, cost_run) where applicable; cf_set_counters(counters, rec_table).  The run then
 * continues bit for bit as the uninterrupted one would (tests/test_gpu_r3.py). */
int cf_set_counters(cf_sim *sim, const uint32_t counters_host[4], const uint32_t *rec_table_dev);

/* Teacher forcing / checkpoint restore of the planning-rollout state: eps [4][MN] (needs noise_beta != 0) and the
 * running cost [MN] (needs cost_on); NULL = keep. */
int cf_set_plan_state(cf_sim *sim, const float *eps_dev, const float *cost_run_dev);

/* Advance n_steps >= 1 physics steps in ONE kernel launch (state in registers across all of them).
 *   cmds_dev     [n_cmds][MN] float4, or [n_ctrl][n_cmds] float4 for CF_CMD_NOMINAL_PLUS_NOISE; n_cmds*cmd_hold >= n_steps
 *   record_every 0: nothing recorded; else see STEP SEMANTICS; record_dev must hold
 *                n_rec = (s0+n_steps)/record_every - s0/record_every slots of D*MN floats (else CF_E_BUFFER). */
int cf_step(cf_sim *sim, const void *cmds_dev, int n_cmds, int cmd_hold,
            int n_steps, int record_every, float *record_dev, size_t record_bytes);

/* The same step driven from HOST buffers (the end-to-end path): copies the commands host->device into staging_dev,
 * runs cf_step recording into staging_dev, copies the records device->host, synchronises the stream.
 * staging_dev must hold cf_staging_bytes(...) bytes (caller-owned device scratch). */
size_t cf_staging_bytes(const cf_sim *sim, int n_cmds, int n_steps, int record_every);
int cf_step_host(cf_sim *sim, const void *cmds_host, int n_cmds, int cmd_hold,
                 int n_steps, int record_every, float *record_host, size_t record_bytes,
                 void *staging_dev, size_t staging_bytes);

/* One fused rollout from HOST buffers with the result copies overlapped -- the planning shape of BASELINE.json configs[2]
 * (every rollout starts from the measured state, only the final state and the minimum distance come
 * back).  Equivalent to  cf_set_state(x0, broadcast) [if x0_host != NULL];  cf_step(cmds, n_cmds, cmd_hold, n_steps,
 * record_every = 0);  cf_get_state_host(state_host);  cf_get_aux_host(CF_AUX_MIN_DIST, min_dist_host)  -- bit-identical
 * results and counters -- but the drones are advanced in n_slices (1..16) consecutive kernel launches over contiguous
 * slices of the batch, and a second stream (owned by the handle, created on first use) copies slice k's rows of the state
 * planes and minimum distances to the host while slice k + 1 computes.
 *   x0_host [D] floats or NULL (keep the current state); cmds_host as cf_step_host; state_host [D][MN] floats;
 *   min_dist_host [MN] floats or NULL (needs obstacles and N = 1: the per-drone read-out of the rollout epilogue, else
 *   CF_E_UNSUPPORTED); staging_dev: cf_staging_bytes(sim, n_cmds, n_steps, 0) + 256 bytes, 256-byte aligned, caller-owned.
 * Host buffers should be pinned (pageable memory serialises the copies).  Synchronises both streams before returning.
 * The copy stream and up to 16 events are created on the first call and owned by the handle (cf_destroy releases them): this
 * is the one place where the library holds CUDA objects of its own; they are internal to the call, which has drained both
 * streams when it returns.  If a slice's launch or copy fails after an earlier slice has run, the planes hold a mixture of
 * advanced and not-advanced drones: the call returns the error, drains both streams and leaves the simulator in the
 * "no state" condition (CF_E_STATE from every stepping call) until cf_reset or cf_set_full(state, ...) gives it one again. */
int cf_rollout_host(cf_sim *sim, const float *x0_host, const void *cmds_host, int n_cmds, int cmd_hold, int n_steps,
                    float *state_host, float *min_dist_host, void *staging_dev, size_t staging_bytes, int n_slices);

/* Copy the state planes [D][MN] to out_dev (device, on the stream) / out_host (host, synchronises). */
int cf_get_state(cf_sim *sim, float *out_dev);
int cf_get_state_host(cf_sim *sim, float *out_host);

/* Auxiliary outputs, see CF_AUX_*.  The _host variant needs device scratch only for CF_AUX_MIN_DIST (M floats). */
int cf_get_aux(cf_sim *sim, int which, void *out_dev);
int cf_get_aux_host(cf_sim *sim, int which, void *out_host, void *scratch_dev, size_t scratch_bytes);

/* Host mirror of the step counter.  It advances with every cf_step CALL; after replaying a captured CUDA graph call
 * cf_sync_counters (synchronises the stream and re-reads the device counter). */
int64_t cf_step_counter(const cf_sim *sim);
int cf_sync_counters(cf_sim *sim);

/* Name of the kernel instantiation the next cf_step would launch and its launch geometry (for profiling notes). */
int cf_describe_launch(const cf_sim *sim, char *buf, size_t buf_len, int *grid, int *block);

/* ---- Sampling-based planner around the planning rollout: hybrid iCEM / MPPI update -------
 * "a hybrid implementation of iCEM and MPPI ..., running five independent controllers in parallel and selecting the
 *  best control sequence at each step.  Following iCEM, each controller truncates the top 1% of trajectories, uses
 *  temporally correlated noise, and warmstarts its sampling from the previous mean solution.  To obtain the mean
 *  across the best samples, we use exponential weighting over all elites, as in MPPI."
 * No equation or parameter is printed; the readings are DESIGN.md R25-R32:
 *   rollout k of controller c applied  u_k[t] = clip(nominal_c[t] + sigma eps_k[t])  (R25, R26) and has cost J_k (R27);
 *   R28 elites E_c = the n_elite rollouts of c with the smallest (J_k as float32 in IEEE total order, NaN last; world index);
 *   R29 w_k = exp(-(J_k - min_E J) / lambda);   R30 mean_c[t] = sum_E w_k u_k[t] / sum_E w_k;
 *   R31 score S_c = sum_E w_k J_k / sum_E w_k, best controller = argmin_c S_c (float32, ties -> lowest c);
 *   R32 plan = mean of the best controller; warm start nominal_c[t] <- mean_c[min(t + shift, H - 1)].
 * The sampled commands are never stored: the update regenerates the elites' commands from the Philox counters.
 * Requirements: N == 1, cmd_source == CF_CMD_NOMINAL_PLUS_NOISE, cost_on, M == n_ctrl * worlds_per_ctrl on this
 * shard (a shard that is to reproduce controllers of a larger run starts at a world_offset that is a multiple of
 * worlds_per_ctrl; nothing else depends on it), and the last calls on sim were a reset / cf_set_state followed by
 * ONE cf_step of horizon * cmd_hold steps with n_cmds == horizon (else CF_E_STATE). */
typedef struct cf_mppi_params {
  uint32_t struct_size;
  int32_t  horizon;      /* H knots */
  int32_t  cmd_hold;     /* physics steps per knot */
  int32_t  n_elite;      /* per controller, 1 .. worlds_per_ctrl (and <= 4096) */
  int32_t  shift;        /* knots executed between two plans (warm-start shift), 0 .. H */
  float    lambda;       /* temperature of the exponential weighting, > 0 */
} cf_mppi_params;
/* layout of info_dev (float32 / int32 words): per controller c: [4c+0] score S_c, [4c+1] J_min, [4c+2] sum of weights,
 * [4c+3] cost of the last elite admitted (threshold); then [4 n_ctrl] = index of the best controller (int32). */
#define CF_MPPI_INFO_WORDS(n_ctrl) (4 * (n_ctrl) + 4)
size_t cf_mppi_scratch_bytes(const cf_sim *sim, const cf_mppi_params *mp);
/* nominal_dev [n_ctrl][H] float4: in = the sequences the rollout was sampled around, out = warm-started sequences;
 * plan_dev [H] float4 (out); info_dev CF_MPPI_INFO_WORDS words (out); elite_idx_dev int32 [n_ctrl][n_elite]
 * (out, may be NULL): world indices local to the controller, ascending; scratch_dev: cf_mppi_scratch_bytes(), 256-byte
 * aligned, caller-owned.  Enqueues on the bound stream. */
int cf_mppi_update(cf_sim *sim, const cf_mppi_params *mp, void *nominal_dev, void *plan_dev, void *info_dev,
                   int32_t *elite_idx_dev, void *scratch_dev, size_t scratch_bytes);
/* cf_mppi_update for callers that have no device memory to give as scratch and no way of getting any.
 * Two kinds of caller are meant.  (1) A planner thread inside a fixed-rate control loop (the 50 Hz loop of
 * PAPER.md:L465-L471): cudaMalloc / cudaFree take driver locks and may synchronise the whole device, so a loop with a
 * deadline must not call them after start-up, and it may not know n_elite / horizon (which size the scratch) before then.
 * (2) A component living inside someone else's process -- a plug-in, or code running under a framework that owns the
 * device's memory pool and hands out fixed input / output buffers only -- which is simply not allowed to allocate.
 * Here the scratch (elite index list, weighted command rows, per-controller means, completion counter) is a fixed
 * CF_MPPI_STATIC_SCRATCH_BYTES array compiled into libcf.so; the caller passes inputs and outputs only, and the call runs
 * no cudaMalloc, cudaFree or other allocating routine.  Results are those of cf_mppi_update (same kernel, same arithmetic).
 *   Limit: cf_mppi_scratch_bytes(sim, mp) <= CF_MPPI_STATIC_SCRATCH_BYTES (8 MiB; BASELINE.json's planner -- 5 controllers,
 *     1000 elites, 25 knots -- needs 2.1 MB), else CF_E_BUFFER with both numbers in cf_last_error(); nothing is launched.
 *   Cost: every GPU whose context loads libcf.so carries the 8 MiB from then until the process exits, used or not.
 *   Set-up: the first call on each device looks up the array's address on THAT device (the device that is current, which
 *     must be the one holding the simulator's workspace: checked, CF_E_ARG otherwise) and keeps it; make that first call
 *     during start-up, outside any stream capture.  Later calls only enqueue a 4-byte memset and the kernel.
 *   Sharing: there is ONE array per device for all simulators, streams and host threads.  It still holds the previous
 *     call's data on entry (the one word that has to start at zero is cleared on the stream by every call), and two calls
 *     whose kernels can overlap on the GPU -- different streams, or different simulators bound to different streams --
 *     overwrite each other's scratch: order them on one stream or with events.  Same-stream calls are safe back to back. */
#define CF_MPPI_STATIC_SCRATCH_BYTES ((size_t)8 << 20)
int cf_mppi_update_static(cf_sim *sim, const cf_mppi_params *mp, void *nominal_dev, void *plan_dev, void *info_dev,
                          int32_t *elite_idx_dev);
/* One planning iteration: cf_set_state(x0_dev [D], broadcast) + cf_step(nominal_dev, H, cmd_hold, H*cmd_hold) +
 * cf_mppi_update(...). */
int cf_mppi_iterate(cf_sim *sim, const cf_mppi_params *mp, const float *x0_dev, void *nominal_dev, void *plan_dev,
                    void *info_dev, int32_t *elite_idx_dev, void *scratch_dev, size_t scratch_bytes);

/* The same iteration driven from HOST buffers (the end-to-end path of a 50 Hz control loop): x0_host [D] is copied
 * host->device, the iteration runs, plan_host [H] float4 and info_host (CF_MPPI_INFO_WORDS words) are copied
 * device->host and the stream is synchronised.  plan_dev / info_dev are device staging as in cf_mppi_iterate. */
int cf_mppi_iterate_host(cf_sim *sim, const cf_mppi_params *mp, const float *x0_host, void *nominal_dev,
                         void *plan_host, void *info_host, void *plan_dev, void *info_dev, void *scratch_dev,
                         size_t scratch_bytes);

/* Selection across shards (multi-GPU: every rank runs its own controllers).
 * cf_mppi_pack_best writes this shard's row  [score S_c of its best controller, c + ctrl_offset (the GLOBAL controller
 * index, as a float), plan (H float4)]  = 2 + 4 H floats to row_dev, from the info_dev / plan_dev of cf_mppi_update.
 * cf_mppi_select reads n_rows such rows (rows_dev [n_rows][2 + 4 H], e.g. an all-gather of every rank's row) and copies the
 * winner to best_row_dev: smallest score compared as a float32 in IEEE total order with NaN last, ties -> smallest global
 * controller index (reading R31) -- the same row on every rank.  Both enqueue on the bound stream. */
#define CF_MPPI_ROW_WORDS(horizon) (2 + 4 * (horizon))
int cf_mppi_pack_best(cf_sim *sim, const cf_mppi_params *mp, const void *info_dev, const void *plan_dev, int ctrl_offset,
                      float *row_dev);
int cf_mppi_select(cf_sim *sim, const float *rows_dev, int n_rows, int horizon, float *best_row_dev);

/* ---- Gradient of a goal distance w.r.t. the command sequence (Fig. 3D) -------------------------
 * "Measuring throughput over ten simulation steps by differentiating a goal distance with respect to the control
 *  inputs"; "differentiating through high-fidelity dynamics, the full onboard controller stack".
 *   L_i = | p_i(after n_steps) - goal |   for every drone i, from the simulator's CURRENT state (which is not modified:
 *   neither the planes nor the step counter), driven by cmds_dev [n_cmds][MN] float4 exactly as cf_step would be;
 *   grad_dev [n_cmds][MN] float4 receives dL_i / d cmds[k][i][0..3]  (commands beyond the last used one: 0);
 *   loss_dev [MN] receives L_i.
 * One hand-written reverse-mode kernel (two launches): forward sweep parking, per step, only what the backward sweep reads
 * non-linearly in scratch_dev (cf_grad_scratch_bytes = (n_steps * HD + 4) * MN floats + 16 bytes, 16-byte aligned; HD = 16 / 18 / 32 for the
 * first-principles model with the rotor / attitude / position interface -- attitude, body rates, rotor speeds, controller
 * integrals, rotor command; position and velocity only when the position controller reads them -- and 8 / 20 for the
 * abstracted model with the attitude / position interface), backward sweep through normalisation, RK4 / Euler, Eqs.
 * (1)-(4), (6) or (7)-(10), mixer, attitude controller and geometric position controller (the full onboard stack of
 * PAPER.md:L69).  Where a clip of the method is active (rotor thrust / speed limits, controller integrals, thrust and tilt
 * limits, rotor-interface command limits) the derivative is taken as 0 (reading R33); the controller tick schedules
 * follow the global step counter.
 * Supported: CF_CMD_BUFFER; every interface of the first-principles model (rotor, torque, attitude, position), attitude
 * and position of the abstracted model; Euler and RK4; per-world randomised parameters.  Configurations with force
 * disturbances (the differentiated rollout draws the same Philox forces as cf_step would from the current
 * step counter), any fidelity extra (full Eq. (6), thrust / torque polynomials incl. the mixer's inverse, Eq. (5), body
 * drag, the simplified abstracted model of PAPER.md:L354) or the torque interface run the GENERAL adjoint kernels: the
 * generic 17 / 13-component pull-back and a full record per step, HD = 32 (first-principles) / 20 (abstracted).  Full
 * Eq. (6) is only piecewise smooth (its coefficients switch with the sign of a rotor's speed error): the gradient is
 * that of the branch taken.  CF_E_UNSUPPORTED: CF_CMD_NOMINAL_PLUS_NOISE (no command buffer to differentiate with respect
 * to).  goal: 3 floats on the HOST.
 * cf_grad_host: the same from HOST buffers -- cmds_host [n_cmds][MN] float4 in, loss_host [MN] and grad_host
 * [n_cmds][MN] float4 out, through staging_dev (cf_grad_staging_bytes(), 256-byte aligned, caller-owned device memory);
 * synchronises the stream. */
size_t cf_grad_scratch_bytes(const cf_sim *sim, int n_steps);
int cf_grad(cf_sim *sim, const void *cmds_dev, int n_cmds, int cmd_hold, int n_steps, const float goal[3],
            float *loss_dev, void *grad_dev, void *scratch_dev, size_t scratch_bytes);
size_t cf_grad_staging_bytes(const cf_sim *sim, int n_cmds);
int cf_grad_host(cf_sim *sim, const void *cmds_host, int n_cmds, int cmd_hold, int n_steps, const float goal[3],
                 float *loss_host, void *grad_host, void *staging_dev, size_t staging_bytes, void *scratch_dev,
                 size_t scratch_bytes);

/* ---- Batched depth ray casting -------------------------------------------------------------
 * "parallel rendering of depth images ... 350k frames per second at a 64x64 ray resolution across 1,024 environments".
 * The paper inherits this from MJX's ray-cast pipeline; its camera model and test scene (MuJoCo XML) are not available, so
 * this is reading R34 on a synthetic scene.  For every drone i (from the CURRENT state planes):
 *   camera origin o = p_i + R_i cam_offset; optical axis = body +x, image right = body -y, image down = body -z;
 *   pixel (row v, column u): d = R_i normalise(1, -(u + 1/2 - W/2) s, -(v + 1/2 - H/2) s),  s = 2 tan(fov_x/2) / W;
 *   depth_dev[i][v][u] = smallest t in (0, t_max] with o + t d on a sphere, an axis-aligned box or the plane z = 0
 *   (distance along the unit ray; a ray starting inside a primitive hits it from the inside), or -1 if there is none.
 * The scene is shared by all worlds.  One kernel launch, thread = ray; arithmetic only (no graphics API). */
#define CF_DEPTH_MAX_PRIMS 32
typedef struct cf_depth_params {
  uint32_t struct_size;
  int32_t  width, height;
  int32_t  n_spheres, n_boxes, ground_plane;
  float    fov_x;                               /* horizontal field of view [rad], (0, 3.1) */
  float    t_max;                               /* <= 0: unlimited */
  float    cam_offset[3];                       /* camera position in the body frame [m] */
  float    spheres[CF_DEPTH_MAX_PRIMS][4];      /* cx cy cz r */
  float    boxes[CF_DEPTH_MAX_PRIMS][6];        /* cx cy cz hx hy hz (half extents) */
} cf_depth_params;
int cf_depth(cf_sim *sim, const cf_depth_params *dp, float *depth_dev /* [MN][height][width] */);
/* The same from HOST buffers: state_host [D][MN] (poses to render; NULL = the simulator's current state) is copied into the
 * state planes, the images go through staging_dev (MN * height * width floats, caller-owned device memory) to depth_host;
 * synchronises the stream. */
int cf_depth_host(cf_sim *sim, const cf_depth_params *dp, const float *state_host, float *depth_host,
                  float *staging_dev, size_t staging_bytes);

const char *cf_last_error(void);
/* Host-side Philox4x32-10 of this library, for the bit-exact check against the oracle's (C9). */
int cf_debug_philox(uint64_t seed, const uint32_t ctr[4], uint32_t out[4]);
/* Device-side Philox4x32-10 + uniform + Box-Muller as the kernels use them: n counters -> n x 4 words, uniforms, normals */
int cf_debug_philox_dev(cf_sim *sim, uint64_t seed, const uint32_t *ctr_dev, int n,
                        uint32_t *words_dev, float *uniform_dev, float *normal_dev);

#ifdef __cplusplus
}
#endif
#endif
