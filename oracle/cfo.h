/* cfo.h -- float64 CPU ORACLE for the Crazyflow batched simulation step.
 *
 * TEST INFRASTRUCTURE ONLY.  This is the plain, slow, obviously-correct restatement of what
 * the hot path computes, written from /root/reference/PAPER.md (Eqs. (1)-(10))
 * and from the readings listed in DESIGN.md ("Readings", mirroring SURVEY.md section 8(c) C0-C12).
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * load it.  It shares no code, header, table or helper with the CUDA path under
 * paper_2606_01478_b200/csrc/ and neither includes the other.
 *
 * Everything is float64 except counters / Philox words (uint32) and the command buffers, which
 * are float32 on purpose: both sides must see bit-identical commands.
 *
 * Layouts (component-major, "planes"):
 *   state  [D][M*N]       D = 17 first-principles: p(0-2) q(3-6, x y z w scalar-last) v(7-9) w(10-12) Omega(13-16, rpm)
 *                         D = 13 abstracted:       p(0-2) Psi(3-5 roll pitch yaw) v(6-8) dPsi(9-11) f_Sigma(12)
 *   ctrl   [14][M*N]      i_R(0-2) i_p(3-5) held attitude cmd(6-9: roll pitch yaw thrust) held rotor cmd(10-13, rpm)
 *   wparam [P][M]         P = 14 FP: m Jx Jy Jz kf0 kf1 kf2 km0 km1 km2 cv_up cv_dn cd_up cd_dn
 *                         P = 11 AB: m a[3] b[3] c[3] c_tau
 *   mind2  [8][M*N]       running minimum of squared centre distance per obstacle
 *   eps    [4][M*N]       AR(1) state of the command noise;  cost_run [M*N] running rollout cost
 *   cmds   [K][M*N][4]    float32 (CMD_BUFFER)  or  [n_ctrl][K][4] nominal sequences (CMD_NOMINAL_PLUS_NOISE)
 *   record [n_rec][D][M*N]
 *
 * Parity pins (tests/test_oracle_pins.py): free fall, hover equilibrium, torque-free precession and
 * conservation laws, quaternion closed form, motor-lag closed forms, mixer round trip, tilted thrust
 * parabola, Eq.(10) linear recurrence, Philox known-answer vectors, distribution moments, brute-force
 * obstacle distance, position/attitude controller special cases, integrator order, fused == split.
 * tests/test_oracle_pins_switches.py: disturbance step (Newton's law on a force-free body: counter, which normals,
 * sigma, world frame, per-world mass, hold over RK4 stages, variance), PARAM slot map of both models one slot at a
 * time, torque interface and thrust-polynomial inverse through the geometry-pinned mixing matrix, simplified
 * abstracted model (Eq. (8) at level attitude with and without Eq. (9)).
 * The controller structure and gains (C5-C7), limits, reset distributions and stream numbering are
 * readings the paper does not print: for those, parity is pinned only by the special cases above.
 */
#ifndef CFO_H
#define CFO_H
#include <stddef.h>
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

enum { CFO_MODEL_FIRST_PRINCIPLES = 0, CFO_MODEL_ABSTRACTED = 1 };
enum { CFO_EULER = 0, CFO_RK4 = 1 };
enum { CFO_IF_ROTOR = 0, CFO_IF_TORQUE = 1, CFO_IF_ATTITUDE = 2, CFO_IF_POSITION = 3 };
enum { CFO_CMD_BUFFER = 0, CFO_CMD_NOMINAL_PLUS_NOISE = 1 };
enum { CFO_AUX_COUNTERS = 0, CFO_AUX_MIN_DIST = 1, CFO_AUX_CTRL = 2, CFO_AUX_WORLD_PARAMS = 3,
       CFO_AUX_REC_TABLE = 4, CFO_AUX_MIN_D2 = 5,
       CFO_AUX_COST = 6,   /* double[MN]: running cost + terminal + obstacle-clearance terms (R27) */
       CFO_AUX_EPS = 7,    /* double[4][MN]: AR(1) noise state, NaN = no command drawn since the last re-arm (R25) */
       CFO_AUX_COST_RUN = 8 /* double[MN]: running part only */ };
#define CFO_REC_TABLE_CAP 4096

typedef struct cfo_params {
  int32_t integrator, iface, cmd_source, ab_thrust_dyn;
  int32_t init_mode;              /* 0 fixed (p = p0_lo, level), 1 box + axis-angle, 2 grid */
  int32_t grid_dims[3];
  int32_t n_obstacles;
  int32_t _pad;
  int64_t world_offset;           /* global index of local world 0 (multi-GPU sharding) */
  double f_phys, f_att, f_pos;
  double mass, J[3], arm, kf[3], km[3], g;
  double cv_up, cv_dn, cd_up, cd_dn;
  double Jp, Ca[3];
  double ab_a[3], ab_b[3], ab_c[3], ab_ctau, ab_cf;
  double rpm_min, rpm_max, thrust_min, thrust_max, tilt_max;
  double kR[3], kW[3], kI[3], iR_max;
  double kp[3], kd[3], ki[3], ip_max[3];
  double rnd_lo[12], rnd_hi[12];
  double dist_sigma;
  double p0_lo[3], p0_hi[3], tilt0_max;
  double grid_spacing, grid_jitter, grid_origin[3];
  double obstacles[8][4];
  double noise_sigma[4], cmd_lo[4], cmd_hi[4];
  /* planning rollouts for the MPPI / iCEM sampler (readings R25-R27) */
  double noise_beta;              /* AR(1) coefficient of the temporally correlated command noise, 0 = white */
  int64_t worlds_per_ctrl;        /* controller of a world = local world index / worlds_per_ctrl (0: one controller) */
  int32_t n_ctrl;                 /* number of nominal sequences in the command buffer [n_ctrl][n_cmds][4] */
  int32_t cost_on;                /* accumulate the running rollout cost */
  double cost_goal[3], cost_w_pos, cost_w_vel, cost_w_term, cost_w_obs, cost_d_safe, cost_w_coll;
} cfo_params;

typedef struct cfo_sim cfo_sim;

void cfo_default_params(cfo_params *p, int model);
int  cfo_state_dim(int model);                 /* 17 / 13 */
int  cfo_world_param_dim(int model);           /* 14 / 11 */
int  cfo_create(cfo_sim **out, int64_t M, int64_t N, int model, const cfo_params *p);
void cfo_destroy(cfo_sim *s);
int  cfo_reset(cfo_sim *s, uint64_t seed);
int  cfo_reset_masked(cfo_sim *s, const uint8_t *mask /* [M] */, uint64_t episode_seed);
int  cfo_set_state(cfo_sim *s, const double *state, int broadcast);
/* teacher forcing: overwrite everything a step depends on (any pointer may be NULL = keep) */
int  cfo_set_full(cfo_sim *s, const double *state, const double *ctrl, const double *wparam,
                  const double *mind2, int64_t step_counter);
int  cfo_set_plan_state(cfo_sim *s, const double *eps, const double *cost_run);
int  cfo_step(cfo_sim *s, const float *cmds, int n_cmds, int cmd_hold, int n_steps, int record_every,
              double *record, size_t record_len /* doubles */);
int  cfo_step_f64cmd(cfo_sim *s, const double *cmds64, int n_cmds, int cmd_hold, int n_steps);
int  cfo_get_state(cfo_sim *s, double *out);
int  cfo_get_aux(cfo_sim *s, int which, void *out);
void cfo_philox(uint64_t seed, const uint32_t ctr[4], uint32_t out[4]);
double cfo_uniform(uint32_t x);
void cfo_normal_pair(uint32_t xa, uint32_t xb, double *z0, double *z1);
/* exposed pieces for pins (single drone, nominal parameters of p) */
void cfo_attitude_tick(const cfo_params *p, const double q[4], const double w[3], const double cmd[4],
                       double iR[3], double eR_out[3], double tau_out[3], double rpm_cmd[4]);
void cfo_position_tick(const cfo_params *p, const double pos[3], const double vel[3], const double zB[3],
                       const double target[4], double ip[3], double att_cmd[4]);
void cfo_mix(const cfo_params *p, const double rpm[4], double *F, double tau[3]);
int  cfo_num_threads(void);
void cfo_set_num_threads(int n);

#ifdef __cplusplus
}
#endif
#endif
