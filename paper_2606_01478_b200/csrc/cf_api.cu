// cf_api.cu -- the C ABI of include/cf.h: argument checking, workspace carving, kernel dispatch, and the small
// non-hot kernels (reset, set_state, minimum-distance read-out, Philox debug).  No device allocation, no CPU path.
#include "../../include/cf.h"
#include "cf_device.cuh"
#include "cf_internal.h"

#include <cstdlib>

#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <new>

using namespace cf;

static thread_local char g_err[512] = "";
char *cf_err_buf() { return g_err; }
extern "C" const char *cf_last_error(void) { return g_err; }
extern "C" int cf_state_dim(int model) { return model == CF_MODEL_FIRST_PRINCIPLES ? 17 : model == CF_MODEL_ABSTRACTED ? 13 : 0; }
extern "C" int cf_world_param_dim(int model) { return model == CF_MODEL_FIRST_PRINCIPLES ? 14 : model == CF_MODEL_ABSTRACTED ? 11 : 0; }

// BASELINE.json:configs[0], configs[2]; limits / gains: DESIGN.md readings R7, R12, R16
extern "C" void cf_default_params(cf_params *p, int model) {
  if (!p) return;
  memset(p, 0, sizeof(*p));
  p->struct_size = (uint32_t)sizeof(cf_params);
  p->integrator = CF_EULER; p->iface = CF_IF_ATTITUDE; p->cmd_source = CF_CMD_BUFFER;
  p->ab_thrust_dyn = 1;
  p->grid_dims[0] = p->grid_dims[1] = p->grid_dims[2] = 1;
  p->f_phys = model == CF_MODEL_FIRST_PRINCIPLES ? 1000.f : 500.f; p->f_att = 500.f; p->f_pos = 100.f;
  p->mass = 0.027f; p->J[0] = 1.395e-5f; p->J[1] = 1.395e-5f; p->J[2] = 2.173e-5f; p->arm = 0.046f;
  p->kf[2] = 3.16e-10f; p->km[2] = 7.94e-12f; p->g = 9.81f;
  p->cv_up = p->cv_dn = (float)(1.0 / 0.03);
  for (int j = 0; j < 3; ++j) { p->ab_a[j] = -130.f; p->ab_b[j] = -16.f; p->ab_c[j] = 130.f; }
  p->ab_ctau = (float)(1.0 / 0.03); p->ab_cf = 1.f;
  p->rpm_min = 0.f; p->rpm_max = 21700.f; p->thrust_min = 0.f; p->thrust_max = 0.55f; p->tilt_max = 0.5f;
  for (int j = 0; j < 3; ++j) { p->kR[j] = 130.f; p->kW[j] = 16.f; }
  p->kI[0] = 20.f; p->kI[1] = 20.f; p->kI[2] = 0.f; p->iR_max = 0.2f;
  p->kp[0] = 8.f; p->kp[1] = 8.f; p->kp[2] = 12.f;
  p->kd[0] = 5.f; p->kd[1] = 5.f; p->kd[2] = 7.f;
  p->ki[0] = 1.f; p->ki[1] = 1.f; p->ki[2] = 6.f;
  p->ip_max[0] = 0.25f; p->ip_max[1] = 0.25f; p->ip_max[2] = 0.4f;
  for (int j = 0; j < 12; ++j) { p->rnd_lo[j] = 1.f; p->rnd_hi[j] = 1.f; }
  p->p0_lo[2] = 1.f; p->p0_hi[2] = 1.f;
  const float pi = 3.14159265358979323846f;
  p->cmd_lo[0] = -0.5f; p->cmd_lo[1] = -0.5f; p->cmd_lo[2] = -pi; p->cmd_lo[3] = 0.05f;
  p->cmd_hi[0] = 0.5f;  p->cmd_hi[1] = 0.5f;  p->cmd_hi[2] = pi;  p->cmd_hi[3] = 0.55f;
  p->n_ctrl = 1;
}

static size_t align256(size_t n) { return (n + 255) & ~(size_t)255; }

struct Carve { size_t state, ctrl, wparam, min_d2, md_drone, eps, cost_run, cost_drone, bcast, counters, rec_table, total; };
static bool wants_eps(const cf_params *p) { return p->cmd_source == CF_CMD_NOMINAL_PLUS_NOISE && p->noise_beta != 0.f; }
static Carve carve(long long M, long long N, int model, const cf_params *p) {
  Carve c;
  size_t MN = (size_t)(M * N), off = 0;
  c.state = off;     off += align256(sizeof(float) * cf_state_dim(model) * MN);
  c.ctrl = off;      off += align256(sizeof(float) * kCtrlPlanes * MN);
  c.wparam = off;    off += align256(sizeof(float) * cf_world_param_dim(model) * (size_t)M);
  c.min_d2 = off;    off += p->n_obstacles > 0 ? align256(sizeof(float) * kMaxObst * MN) : 0;
  c.md_drone = off;  off += p->n_obstacles > 0 ? align256(sizeof(float) * MN) : 0;
  c.eps = off;       off += wants_eps(p) ? align256(sizeof(float) * 4 * MN) : 0;
  c.cost_run = off;  off += p->cost_on ? align256(sizeof(float) * MN) : 0;
  c.cost_drone = off; off += p->cost_on ? align256(sizeof(float) * MN) : 0;
  c.bcast = off;     off += 256;
  c.counters = off;  off += align256(sizeof(Counters));
  c.rec_table = off; off += align256(sizeof(uint32_t) * kRecTableCap);
  c.total = off;
  return c;
}

static int validate(long long M, long long N, int model, const cf_params *p) {
  if (!p) return fail(CF_E_ARG, "params is NULL");
  if (p->struct_size != sizeof(cf_params))
    return fail(CF_E_ARG, "cf_params.struct_size %u != %zu", p->struct_size, sizeof(cf_params));
  if (model != CF_MODEL_FIRST_PRINCIPLES && model != CF_MODEL_ABSTRACTED) return fail(CF_E_ARG, "bad model %d", model);
  if (M < 1 || N < 1) return fail(CF_E_ARG, "M and N must be >= 1");
  if (M > ((long long)1 << 31) || N > ((long long)1 << 31) || M * N >= ((long long)1 << 31))
    return fail(CF_E_SHAPE, "M*N must be < 2^31");
  if (p->integrator != CF_EULER && p->integrator != CF_RK4) return fail(CF_E_ARG, "bad integrator");
  if (p->iface < CF_IF_ROTOR || p->iface > CF_IF_POSITION) return fail(CF_E_ARG, "bad iface");
  if (p->cmd_source != CF_CMD_BUFFER && p->cmd_source != CF_CMD_NOMINAL_PLUS_NOISE) return fail(CF_E_ARG, "bad cmd_source");
  if (!(p->f_phys > 0) || !(p->f_att > 0) || !(p->f_pos > 0)) return fail(CF_E_ARG, "rates must be > 0");
  double ad = (double)p->f_phys / p->f_att, pd = (double)p->f_phys / p->f_pos;
  if (ad < 1 || pd < 1 || ad != std::floor(ad) || pd != std::floor(pd))
    return fail(CF_E_SHAPE, "f_phys/f_att and f_phys/f_pos must be integers >= 1");
  if (model == CF_MODEL_ABSTRACTED && p->iface != CF_IF_ATTITUDE && p->iface != CF_IF_POSITION)
    return fail(CF_E_UNSUPPORTED, "the abstracted model interfaces at the attitude or position level only");
  if (p->n_obstacles < 0 || p->n_obstacles > CF_MAX_OBSTACLES) return fail(CF_E_ARG, "n_obstacles out of range");
  if (p->init_mode < 0 || p->init_mode > 2) return fail(CF_E_ARG, "bad init_mode");
  if (p->init_mode == 2 && (p->grid_dims[0] < 1 || p->grid_dims[1] < 1)) return fail(CF_E_ARG, "bad grid_dims");
  if (!(p->mass > 0) || !(p->J[0] > 0) || !(p->J[1] > 0) || !(p->J[2] > 0)) return fail(CF_E_ARG, "mass/J must be > 0");
  if (model == CF_MODEL_FIRST_PRINCIPLES && p->iface != CF_IF_ROTOR && !(p->kf[2] > 0))
    return fail(CF_E_ARG, "controller needs kf[2] > 0");
  if (!(p->noise_beta >= 0.f && p->noise_beta < 1.f)) return fail(CF_E_ARG, "noise_beta must be in [0, 1)");
  if (p->n_ctrl < 1 || p->worlds_per_ctrl < 0) return fail(CF_E_ARG, "n_ctrl >= 1 and worlds_per_ctrl >= 0");
  if (p->cmd_source == CF_CMD_NOMINAL_PLUS_NOISE && p->worlds_per_ctrl > 0 &&
      (M - 1) / p->worlds_per_ctrl >= p->n_ctrl)
    return fail(CF_E_SHAPE, "%lld worlds need more than n_ctrl = %d nominal sequences", (long long)M, p->n_ctrl);
  if (p->cost_on && N != 1) return fail(CF_E_UNSUPPORTED, "the rollout cost needs N == 1");
  if (p->world_offset < 0 || p->world_offset + M > ((long long)1 << 32)) return fail(CF_E_SHAPE, "world_offset out of range");
  for (int j = 0; j < 12; ++j) {
    if (!(p->rnd_lo[j] <= p->rnd_hi[j])) return fail(CF_E_ARG, "rnd_lo[%d] > rnd_hi[%d] (or NaN)", j, j);
    // slots the kernels take reciprocals of: mass and inertia (both models: slot 0; FP: 1-3), motor time constant (FP: 6)
    bool divides = j == 0 || (model == CF_MODEL_FIRST_PRINCIPLES && (j <= 3 || j == 6));
    if (divides && !(p->rnd_lo[j] > 0.f)) return fail(CF_E_ARG, "rnd_lo[%d] must be > 0 (the slot is divided by)", j);
  }
  for (int j = 0; j < 4; ++j) {
    if (!(p->cmd_lo[j] <= p->cmd_hi[j])) return fail(CF_E_ARG, "cmd_lo[%d] > cmd_hi[%d] (or NaN)", j, j);
    if (!(p->noise_sigma[j] >= 0.f)) return fail(CF_E_ARG, "noise_sigma[%d] must be >= 0", j);
  }
  if (!(p->dist_sigma >= 0.f)) return fail(CF_E_ARG, "dist_sigma must be >= 0");
  return CF_OK;
}

extern "C" size_t cf_workspace_bytes(int64_t M, int64_t N, int model, const cf_params *p) {
  if (validate(M, N, model, p) != CF_OK) return 0;
  return carve(M, N, model, p).total;
}

static double hover_rpm_nominal(const cf_params *p) {
  double f = (double)p->mass * p->g / 4.0, k0 = p->kf[0], k1 = p->kf[1], k2 = p->kf[2];
  if (!(k2 > 0)) return 0.0;
  if (k0 == 0 && k1 == 0) return std::sqrt(f / k2);
  double disc = k1 * k1 - 4 * k2 * (k0 - f);
  return (-k1 + std::sqrt(disc > 0 ? disc : 0)) / (2 * k2);
}

static void fill_dev_params(cf_sim *s) {
  const cf_params &p = s->p;
  DevParams &d = s->dp;
  memset(&d, 0, sizeof(d));
  double h = 1.0 / p.f_phys;
  d.att_div = (int)std::llround((double)p.f_phys / p.f_att);
  d.pos_div = (int)std::llround((double)p.f_phys / p.f_pos);
  d.h = (float)h; d.half_h = (float)(0.5 * h); d.h_sixth = (float)(h / 6.0);
  d.h_att = (float)(d.att_div * h); d.h_pos = (float)(d.pos_div * h); d.g = p.g;
  d.mass = p.mass; d.inv_mass = (float)(1.0 / p.mass);
  double lever = (double)p.arm / std::sqrt(2.0);      // reading R6: arm is centre-to-rotor, X configuration
  d.lever = (float)lever;
  for (int j = 0; j < 3; ++j) {
    d.J[j] = p.J[j]; d.inv_J[j] = (float)(1.0 / p.J[j]); d.kf[j] = p.kf[j]; d.km[j] = p.km[j]; d.Ca[j] = p.Ca[j];
    d.ab_a[j] = p.ab_a[j]; d.ab_b[j] = p.ab_b[j]; d.ab_c[j] = p.ab_c[j];
    d.kR[j] = p.kR[j]; d.kW[j] = p.kW[j]; d.kI[j] = p.kI[j]; d.Jnom[j] = p.J[j];
    d.kp[j] = p.kp[j]; d.kd[j] = p.kd[j]; d.ki[j] = p.ki[j]; d.ip_max[j] = p.ip_max[j];
  }
  d.cv_up = p.cv_up; d.cv_dn = p.cv_dn; d.cd_up = p.cd_up; d.cd_dn = p.cd_dn;
  d.Jp_rad = (float)((double)p.Jp * 2.0 * 3.14159265358979323846 / 60.0);
  d.ab_ctau = p.ab_ctau; d.ab_cf = p.ab_cf; d.ab_thrust_dyn = p.ab_thrust_dyn;
  d.thrust_poly = (p.kf[0] != 0.f || p.kf[1] != 0.f);
  {   // bound constants of the abstracted model's angle recursion over every world this simulator can hold (slot map of
      // reset_params_kernel: a_j <- fac[1 + j], b_j <- fac[4 + j]), rounded up by 1e-6 relative
    double ha = 0, hb1 = 0;
    for (int j = 0; j < 3; ++j) {
      ha = std::max(ha, h * std::fabs((double)p.ab_a[j]) * std::max(std::fabs((double)p.rnd_lo[1 + j]), std::fabs((double)p.rnd_hi[1 + j])));
      hb1 = std::max(hb1, std::max(std::fabs(1.0 + h * p.ab_b[j] * p.rnd_lo[4 + j]), std::fabs(1.0 + h * p.ab_b[j] * p.rnd_hi[4 + j])));
    }
    d.bnd_ha = (float)(ha * (1.0 + 1e-6)); d.bnd_hb1 = (float)(hb1 * (1.0 + 1e-6));
  }
  d.has_drag = (p.Ca[0] != 0.f || p.Ca[1] != 0.f || p.Ca[2] != 0.f);
  d.has_gyro = p.Jp != 0.f;
  d.inv_4lever = (float)(1.0 / (4.0 * lever));
  if (p.kf[2] > 0) {
    double kappa = (double)p.km[2] / p.kf[2];
    d.inv_4kappa = kappa != 0 ? (float)(1.0 / (4.0 * kappa)) : 0.f;
    d.inv_kf2 = (float)(1.0 / p.kf[2]);
  }
  d.f_rotor_max = (float)((double)p.kf[0] + (double)p.kf[1] * p.rpm_max + (double)p.kf[2] * p.rpm_max * p.rpm_max);
  d.rpm_min = p.rpm_min; d.rpm_max = p.rpm_max; d.thrust_min = p.thrust_min; d.thrust_max = p.thrust_max;
  d.tilt_max = p.tilt_max; d.iR_max = p.iR_max; d.dist_sigma = p.dist_sigma; d.n_obst = p.n_obstacles;
  d.use_noise = p.cmd_source == CF_CMD_NOMINAL_PLUS_NOISE;
  d.hover_thrust = (float)((double)p.mass * p.g);
  d.hover_rpm = s->model == CF_MODEL_FIRST_PRINCIPLES ? (float)hover_rpm_nominal(&p) : 0.f;
  for (int j = 0; j < kMaxObst; ++j) {
    for (int k = 0; k < 4; ++k) d.obst[j][k] = p.obstacles[j][k];
    if (j < p.n_obstacles) {
      double cx = p.obstacles[j][0], cy = p.obstacles[j][1], cz = p.obstacles[j][2];
      d.obst_q[j] = make_float4((float)(-2 * cx), (float)(-2 * cy), (float)(-2 * cz), (float)(cx * cx + cy * cy + cz * cz));
    } else {
      d.obst_q[j] = make_float4(0.f, 0.f, 0.f, INFINITY);
    }
    d.obst_x[j] = d.obst_q[j].x; d.obst_y[j] = d.obst_q[j].y; d.obst_z[j] = d.obst_q[j].z;
  }
  for (int k = 0; k < 4; ++k) { d.noise_sigma[k] = p.noise_sigma[k]; d.cmd_lo[k] = p.cmd_lo[k]; d.cmd_hi[k] = p.cmd_hi[k]; }
  d.noise_beta = p.noise_beta; d.noise_gain = (float)std::sqrt(1.0 - (double)p.noise_beta * p.noise_beta);
  for (int k = 0; k < 3; ++k) d.cost_goal[k] = p.cost_goal[k];
  d.cost_hw_pos = (float)(h * p.cost_w_pos); d.cost_hw_vel = (float)(h * p.cost_w_vel);
  d.cost_w_term = p.cost_w_term; d.cost_w_obs = p.cost_w_obs; d.cost_d_safe = p.cost_d_safe; d.cost_w_coll = p.cost_w_coll;
  d.cost_on = p.cost_on;
}

static int needed_opt(const cf_sim *s) {
  const cf_params &p = s->p;
  int opt = 0;
  for (int j = 0; j < 12; ++j) if (p.rnd_lo[j] != 1.f || p.rnd_hi[j] != 1.f) opt |= OPT_RANDP;
  if (p.dist_sigma > 0.f) opt |= OPT_DIST;
  if (p.n_obstacles > 0) opt |= OPT_OBST;
  if (p.cmd_source == CF_CMD_NOMINAL_PLUS_NOISE) opt |= OPT_NOISE;
  if (wants_eps(&p)) opt |= OPT_AR;
  if (p.cost_on) opt |= OPT_COST;
  bool extras = p.Jp != 0.f || p.Ca[0] != 0.f || p.Ca[1] != 0.f || p.Ca[2] != 0.f;
  if (s->model == CF_MODEL_FIRST_PRINCIPLES)
    extras = extras || p.cv_up != p.cv_dn || p.cd_up != 0.f || p.cd_dn != 0.f || p.kf[0] != 0.f || p.kf[1] != 0.f ||
             p.km[0] != 0.f || p.km[1] != 0.f;
  else
    extras = extras || !p.ab_thrust_dyn;
  if (extras) opt |= OPT_EXTRAS;
  return opt;
}

// ---------------------------------------------------------------------------------------------------------------
// Reset kernels (C9): PARAM stream -> per-world plant parameters, INIT stream -> initial state.
struct ResetArgs {
  float rnd_lo[12], rnd_hi[12];
  float nominal[14];                 // nominal world-parameter row (FP: 14, AB: 11 used)
  float p0_lo[3], p0_hi[3], tilt0_max, grid_spacing, grid_jitter, grid_origin[3];
  int grid_dims[3], init_mode, model;
  float hover_rpm, hover_thrust;
  long long M, N, MN, world_offset;
  uint32_t seed_lo, seed_hi;
};

__global__ void reset_params_kernel(float *wparam, const __grid_constant__ ResetArgs R) {
  long long w = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (w >= R.M) return;
  uint32_t wg = (uint32_t)(w + R.world_offset);
  float fac[12];
#pragma unroll
  for (int b = 0; b < 3; ++b) {
    uint32_t r[4];
    philox4x32_10(R.seed_lo, R.seed_hi, wg, 0u, (uint32_t)b, STREAM_PARAM, r);
#pragma unroll
    for (int k = 0; k < 4; ++k) fac[4 * b + k] = R.rnd_lo[4 * b + k] + (R.rnd_hi[4 * b + k] - R.rnd_lo[4 * b + k]) * u01(r[k]);
  }
  const long long M = R.M;
  if (R.model == MODEL_FP) {   // reading R17: slots (m, Jx, Jy, Jz | k_f, k_m, tau_m, -)
    wparam[w] = R.nominal[0] * fac[0];
    for (int j = 0; j < 3; ++j) wparam[(1 + j) * M + w] = R.nominal[1 + j] * fac[1 + j];
    for (int j = 0; j < 3; ++j) wparam[(4 + j) * M + w] = R.nominal[4 + j] * fac[4];
    for (int j = 0; j < 3; ++j) wparam[(7 + j) * M + w] = R.nominal[7 + j] * fac[5];
    for (int j = 0; j < 4; ++j) wparam[(10 + j) * M + w] = R.nominal[10 + j] / fac[6];
  } else {                     // slots (m, a[3] | b[3], - | c[3], c_tau)
    wparam[w] = R.nominal[0] * fac[0];
    for (int j = 0; j < 3; ++j) wparam[(1 + j) * M + w] = R.nominal[1 + j] * fac[1 + j];
    for (int j = 0; j < 3; ++j) wparam[(4 + j) * M + w] = R.nominal[4 + j] * fac[4 + j];
    for (int j = 0; j < 3; ++j) wparam[(7 + j) * M + w] = R.nominal[7 + j] * fac[8 + j];
    wparam[10 * M + w] = R.nominal[10] * fac[11];
  }
}

// controller integrals 0, held commands = hover of the nominal model, min distance +inf (reading R20)
struct RearmPlanes { float *ctrl, *min_d2, *eps, *cost_run; };
__device__ __forceinline__ void rearm(const RearmPlanes &rp, long long MN, long long i, float hover_rpm,
                                      float hover_thrust) {
  float *ctrl = rp.ctrl, *min_d2 = rp.min_d2;
  if (rp.eps) rp.eps[i] = __int_as_float(0x7fc00000);      // R25: NaN in plane 0 = the next command starts a fresh chain
  if (rp.cost_run) rp.cost_run[i] = 0.f;                   // R27
#pragma unroll
  for (int c = 0; c < 9; ++c) ctrl[c * MN + i] = 0.f;
  ctrl[9 * MN + i] = hover_thrust;
#pragma unroll
  for (int k = 0; k < 4; ++k) ctrl[(10 + k) * MN + i] = hover_rpm;
  if (min_d2) {
#pragma unroll
    for (int j = 0; j < kMaxObst; ++j) min_d2[j * MN + i] = __int_as_float(0x7f800000);
  }
}

__global__ void reset_state_kernel(float *state, RearmPlanes rp, const uint8_t *mask, const __grid_constant__ ResetArgs R) {
  long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= R.MN) return;
  long long w = i / R.N, n = i - w * R.N;
  if (mask != nullptr && mask[w] == 0) return;             // cf_reset_masked: this world keeps running
  uint32_t wg = (uint32_t)(w + R.world_offset), nn = (uint32_t)n;
  float pos[3], q[4] = { 0.f, 0.f, 0.f, 1.f };
  uint32_t r[4];
  if (R.init_mode == 0) {
    for (int j = 0; j < 3; ++j) pos[j] = R.p0_lo[j];
  } else if (R.init_mode == 1) {
    philox4x32_10(R.seed_lo, R.seed_hi, wg, nn, 0u, STREAM_INIT, r);
    for (int j = 0; j < 3; ++j) pos[j] = R.p0_lo[j] + (R.p0_hi[j] - R.p0_lo[j]) * u01(r[j]);
    philox4x32_10(R.seed_lo, R.seed_hi, wg, nn, 1u, STREAM_INIT, r);      // reading R19
    float zeta = 2.f * u01(r[0]) - 1.f, theta = R.tilt0_max * u01(r[2]);
    float sa, ca, sh, ch;
    sincospif(2.f * u01(r[1]), &sa, &ca);
    float sxy = sqrtf(fmaxf(1.f - zeta * zeta, 0.f));
    sincosf(0.5f * theta, &sh, &ch);
    q[0] = sxy * ca * sh; q[1] = sxy * sa * sh; q[2] = zeta * sh; q[3] = ch;
  } else {
    philox4x32_10(R.seed_lo, R.seed_hi, wg, nn, 0u, STREAM_INIT, r);
    long long gx = R.grid_dims[0], gy = R.grid_dims[1];
    long long cell[3] = { n % gx, (n / gx) % gy, n / (gx * gy) };
    for (int j = 0; j < 3; ++j)
      pos[j] = R.grid_origin[j] + R.grid_spacing * (float)cell[j] + R.grid_jitter * (2.f * u01(r[j]) - 1.f);
  }
  const long long MN = R.MN;
  const int D = R.model == MODEL_FP ? 17 : 13;
  for (int j = 0; j < D; ++j) state[j * MN + i] = 0.f;
  for (int j = 0; j < 3; ++j) state[j * MN + i] = pos[j];
  if (R.model == MODEL_FP) {
    for (int j = 0; j < 4; ++j) state[(3 + j) * MN + i] = q[j];
    for (int k = 0; k < 4; ++k) state[(13 + k) * MN + i] = R.hover_rpm;
  } else {
    float Rm[3][3];
    quat_to_R(q, Rm);
    state[3 * MN + i] = atan2f(Rm[2][1], Rm[2][2]);
    state[4 * MN + i] = -asinf(clipf(Rm[2][0], -1.f, 1.f));
    state[5 * MN + i] = atan2f(Rm[1][0], Rm[0][0]);
    state[12 * MN + i] = R.hover_thrust;
  }
  rearm(rp, MN, i, R.model == MODEL_FP ? R.hover_rpm : 0.f, R.hover_thrust);
}

__global__ void set_state_kernel(float *state, RearmPlanes rp, const float *src, int broadcast, int D,
                                 long long MN, float hover_rpm, float hover_thrust) {
  long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= MN) return;
  for (int j = 0; j < D; ++j) state[j * MN + i] = broadcast ? src[j] : src[j * MN + i];
  rearm(rp, MN, i, hover_rpm, hover_thrust);
}

__global__ void set_counters_kernel(Counters *c, uint32_t s, int zero_rest) {
  c->s = s;
  if (zero_rest) { c->att_ticks = 0; c->pos_ticks = 0; c->n_rec_total = 0; }
  c->blocks_done = 0;
}

__global__ void set_counters4_kernel(Counters *c, uint32_t s, uint32_t att, uint32_t pos, uint32_t n_rec) {
  c->s = s; c->att_ticks = att; c->pos_ticks = pos; c->n_rec_total = n_rec;
  c->blocks_done = 0;
}

// CF_AUX_NONFINITE: out[0] = number of drones with a NaN / Inf in any state component, out[1] = the first such drone
__global__ void nonfinite_init_kernel(uint32_t *out) { out[0] = 0u; out[1] = 0xFFFFFFFFu; }
__global__ void nonfinite_kernel(const float *state, int D, long long MN, uint32_t *out) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  bool bad = false;
  if (i < MN)
    for (int d = 0; d < D; ++d) bad |= !isfinite(state[(long long)d * MN + i]);
  const unsigned m = __ballot_sync(0xffffffffu, bad);
  if (m && (threadIdx.x & 31) == 0) {
    atomicAdd(out, (uint32_t)__popc(m));
    atomicMin(out + 1, (uint32_t)(i + __ffs(m) - 1));
  }
}

// C10: per world, min over drones, obstacles (and, through min_d2, steps) of |p - c_j| - r_j.  One warp per world.
__global__ void min_dist_kernel(const float *min_d2, float *out, long long M, long long N, long long MN,
                                const __grid_constant__ DevParams P) {
  long long w = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  int lane = threadIdx.x & 31;
  if (w >= M) return;
  float best = __int_as_float(0x7f800000);
  for (long long n = lane; n < N; n += 32) {
    for (int j = 0; j < P.n_obst; ++j) best = fminf(best, sqrtf(min_d2[j * MN + w * N + n]) - P.obst[j][3]);
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) best = fminf(best, __shfl_xor_sync(0xffffffffu, best, o));
  if (lane == 0) out[w] = best;
}

// N small (single drone per world): one thread per world, coalesced over worlds
__global__ void min_dist_small_n_kernel(const float *min_d2, float *out, long long M, long long N, long long MN,
                                        const __grid_constant__ DevParams P) {
  long long w = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (w >= M) return;
  float best = __int_as_float(0x7f800000);
  for (long long n = 0; n < N; ++n) {
#pragma unroll
    for (int j = 0; j < kMaxObst; ++j)
      if (j < P.n_obst) best = fminf(best, sqrtf(min_d2[j * MN + w * N + n]) - P.obst[j][3]);
  }
  out[w] = best;
}

// R27 read-out outside the rollout epilogue (after cf_set_state / cf_set_full): same terms, from the planes
__global__ void cost_readout_kernel(const float *state, const float *min_d2, const float *cost_run, float *out,
                                    long long MN, const __grid_constant__ DevParams P) {
  long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= MN) return;
  float d_min = __int_as_float(0x7f800000);
  if (min_d2) {
#pragma unroll
    for (int j = 0; j < kMaxObst; ++j)
      if (j < P.n_obst) d_min = fminf(d_min, sqrtf(min_d2[j * MN + i]) - P.obst[j][3]);
  }
  float ex = state[i] - P.cost_goal[0], ey = state[MN + i] - P.cost_goal[1], ez = state[2 * MN + i] - P.cost_goal[2];
  float J = fmaf(P.cost_w_term, fmaf(ez, ez, fmaf(ey, ey, ex * ex)), cost_run[i]);
  float gap = P.cost_d_safe - d_min;
  if (gap > 0.0f) J = fmaf(P.cost_w_obs * gap, gap, J);
  if (d_min < 0.0f) J += P.cost_w_coll;
  out[i] = J;
}

__global__ void philox_debug_kernel(uint32_t seed_lo, uint32_t seed_hi, const uint32_t *ctr, int n, uint32_t *words,
                                    float *uni, float *nrm) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  uint32_t r[4];
  philox4x32_10(seed_lo, seed_hi, ctr[4 * i], ctr[4 * i + 1], ctr[4 * i + 2], ctr[4 * i + 3], r);
  float z[4];
  normal_pair(r[0], r[1], z[0], z[1]);
  normal_pair(r[2], r[3], z[2], z[3]);
  for (int k = 0; k < 4; ++k) {
    if (words) words[4 * i + k] = r[k];
    if (uni) uni[4 * i + k] = u01(r[k]);
    if (nrm) nrm[4 * i + k] = z[k];
  }
}

// ---------------------------------------------------------------------------------------------------------------
extern "C" int cf_create(cf_sim **out, int64_t M, int64_t N, int model, const cf_params *p, void *workspace_dev,
                         size_t workspace_bytes) {
  if (!out) return fail(CF_E_ARG, "out is NULL");
  *out = nullptr;
  int rc = validate(M, N, model, p);
  if (rc != CF_OK) return rc;
  Carve c = carve(M, N, model, p);
  if (!workspace_dev) return fail(CF_E_ARG, "workspace_dev is NULL");
  if (((uintptr_t)workspace_dev & 255) != 0) return fail(CF_E_BUFFER, "workspace must be 256-byte aligned");
  if (workspace_bytes < c.total) return fail(CF_E_BUFFER, "workspace too small: %zu < %zu", workspace_bytes, c.total);
  cf_sim *s = new (std::nothrow) cf_sim();
  if (!s) return fail(CF_E_ARG, "out of host memory");
  s->M = M; s->N = N; s->MN = M * N; s->model = model; s->D = cf_state_dim(model); s->P = cf_world_param_dim(model);
  s->p = *p;
  char *base = (char *)workspace_dev;
  s->state = (float *)(base + c.state); s->ctrl = (float *)(base + c.ctrl); s->wparam = (float *)(base + c.wparam);
  s->min_d2 = p->n_obstacles > 0 ? (float *)(base + c.min_d2) : nullptr;
  s->md_drone = p->n_obstacles > 0 ? (float *)(base + c.md_drone) : nullptr;
  s->bcast_buf = (float *)(base + c.bcast);
  s->eps = wants_eps(p) ? (float *)(base + c.eps) : nullptr;
  s->cost_run = p->cost_on ? (float *)(base + c.cost_run) : nullptr;
  s->cost_drone = p->cost_on ? (float *)(base + c.cost_drone) : nullptr;
  s->cost_valid = false; s->rearmed = false; s->last_fresh = false; s->last_s0 = 0; s->last_n_steps = s->last_n_cmds = s->last_cmd_hold = 0;
  s->pending_bcast = false; s->md_valid = false;
  s->counters = (Counters *)(base + c.counters); s->rec_table = (uint32_t *)(base + c.rec_table);
  s->last_rec_mode = REC_NONE; s->last_rec_heavy = false;
  s->stream = 0; s->seed = 0; s->s_host = 0; s->n_rec_host = 0; s->have_state = false;
  s->hover_rpm = (float)hover_rpm_nominal(p);
  fill_dev_params(s);
  s->opt = needed_opt(s);
  const char *name = nullptr;
  bool ok = model == CF_MODEL_FIRST_PRINCIPLES
      ? launch_fp(p->integrator, p->iface, s->opt, REC_NONE, nullptr, nullptr, nullptr, &name, nullptr, true)
      : launch_ab(p->integrator, p->iface, s->opt, REC_NONE, nullptr, nullptr, nullptr, &name, nullptr, true);
  if (!ok) { delete s; return fail(CF_E_UNSUPPORTED, "no kernel instantiation for this configuration"); }
  { const char *fg = getenv("CF_FORCE_GENERAL"); s->force_general = fg && fg[0] == '1'; }
  *out = s;
  return CF_OK;
}

extern "C" int cf_destroy(cf_sim *sim) {
  if (!sim) return fail(CF_E_ARG, "sim is NULL");
  for (cudaEvent_t e : sim->slice_ev) if (e) cudaEventDestroy(e);
  if (sim->copy_stream && sim->copy_stream_owned) cudaStreamDestroy(sim->copy_stream);
  delete sim;
  return CF_OK;
}

extern "C" int cf_set_stream(cf_sim *sim, void *cuda_stream) {
  if (!sim) return fail(CF_E_ARG, "sim is NULL");
  sim->stream = (cudaStream_t)cuda_stream;
  return CF_OK;
}

extern "C" int cf_set_copy_stream(cf_sim *sim, void *cuda_stream) {
  if (!sim) return fail(CF_E_ARG, "sim is NULL");
  if (sim->copy_stream && sim->copy_stream_owned) CF_CUDA(cudaStreamDestroy(sim->copy_stream));
  sim->copy_stream = (cudaStream_t)cuda_stream;      // NULL: cf_rollout_host creates its own on the next call
  sim->copy_stream_owned = false;
  return CF_OK;
}

static int grid_for(long long n, int block) { return (int)((n + block - 1) / block); }
static RearmPlanes rearm_planes(const cf_sim *sim) { return RearmPlanes{ sim->ctrl, sim->min_d2, sim->eps, sim->cost_run }; }

static void fill_reset_args(const cf_sim *sim, uint64_t seed, ResetArgs &R) {
  const cf_params &p = sim->p;
  memset(&R, 0, sizeof(R));
  for (int j = 0; j < 12; ++j) { R.rnd_lo[j] = p.rnd_lo[j]; R.rnd_hi[j] = p.rnd_hi[j]; }
  if (sim->model == CF_MODEL_FIRST_PRINCIPLES) {
    R.nominal[0] = p.mass;
    for (int j = 0; j < 3; ++j) { R.nominal[1 + j] = p.J[j]; R.nominal[4 + j] = p.kf[j]; R.nominal[7 + j] = p.km[j]; }
    R.nominal[10] = p.cv_up; R.nominal[11] = p.cv_dn; R.nominal[12] = p.cd_up; R.nominal[13] = p.cd_dn;
  } else {
    R.nominal[0] = p.mass;
    for (int j = 0; j < 3; ++j) { R.nominal[1 + j] = p.ab_a[j]; R.nominal[4 + j] = p.ab_b[j]; R.nominal[7 + j] = p.ab_c[j]; }
    R.nominal[10] = p.ab_ctau;
  }
  for (int j = 0; j < 3; ++j) {
    R.p0_lo[j] = p.p0_lo[j]; R.p0_hi[j] = p.p0_hi[j]; R.grid_origin[j] = p.grid_origin[j]; R.grid_dims[j] = p.grid_dims[j];
  }
  R.tilt0_max = p.tilt0_max; R.grid_spacing = p.grid_spacing; R.grid_jitter = p.grid_jitter;
  R.init_mode = p.init_mode; R.model = sim->model;
  R.hover_rpm = sim->hover_rpm; R.hover_thrust = (float)((double)p.mass * p.g);
  R.M = sim->M; R.N = sim->N; R.MN = sim->MN; R.world_offset = p.world_offset;
  R.seed_lo = (uint32_t)(seed & 0xFFFFFFFFu); R.seed_hi = (uint32_t)(seed >> 32);
}

extern "C" int cf_reset(cf_sim *sim, uint64_t seed) {
  if (!sim) return fail(CF_E_ARG, "sim is NULL");
  ResetArgs R;
  fill_reset_args(sim, seed, R);
  reset_params_kernel<<<grid_for(sim->M, 128), 128, 0, sim->stream>>>(sim->wparam, R);
  reset_state_kernel<<<grid_for(sim->MN, 128), 128, 0, sim->stream>>>(sim->state, rearm_planes(sim), nullptr, R);
  set_counters_kernel<<<1, 1, 0, sim->stream>>>(sim->counters, 0u, 1);
  CF_CUDA(cudaMemsetAsync(sim->rec_table, 0, sizeof(uint32_t) * kRecTableCap, sim->stream));
  CF_CUDA(cudaGetLastError());
  sim->seed = seed; sim->s_host = 0; sim->n_rec_host = 0; sim->have_state = true; sim->wparam_foreign = false;
  sim->pending_bcast = false; sim->md_valid = false; sim->cost_valid = false; sim->rearmed = true;
  return CF_OK;
}

extern "C" int cf_reset_masked(cf_sim *sim, const uint8_t *mask_dev, uint64_t episode_seed) {
  if (!sim || !mask_dev) return fail(CF_E_ARG, "NULL argument");
  if (!sim->have_state) return fail(CF_E_STATE, "cf_reset_masked needs a prior cf_reset (world parameters)");
  { int rc = cf_materialise(sim); if (rc != CF_OK) return rc; }
  ResetArgs R;
  fill_reset_args(sim, episode_seed, R);
  reset_state_kernel<<<grid_for(sim->MN, 128), 128, 0, sim->stream>>>(sim->state, rearm_planes(sim), mask_dev, R);
  CF_CUDA(cudaGetLastError());
  sim->md_valid = false; sim->cost_valid = false; sim->rearmed = false;
  return CF_OK;
}

static int launch_set_state(cf_sim *sim, const float *src, int broadcast) {
  float hover_thrust = (float)((double)sim->p.mass * sim->p.g);
  set_state_kernel<<<grid_for(sim->MN, 128), 128, 0, sim->stream>>>(
      sim->state, rearm_planes(sim), src, broadcast, sim->D, sim->MN,
      sim->model == CF_MODEL_FIRST_PRINCIPLES ? sim->hover_rpm : 0.f, hover_thrust);
  CF_CUDA(cudaGetLastError());
  return CF_OK;
}

// A broadcast cf_set_state is lazy: the D floats are parked in the workspace and the next cf_step starts every drone
// from them in registers (no 35-plane write + re-read).  Anything else that touches the planes materialises it first.
static int materialise(cf_sim *sim);
int cf_materialise(cf_sim *sim) { return materialise(sim); }
static int materialise(cf_sim *sim) {
  if (!sim->pending_bcast) return CF_OK;
  sim->pending_bcast = false;
  return launch_set_state(sim, sim->bcast_buf, 1);
}

extern "C" int cf_set_state(cf_sim *sim, const float *state_dev, int broadcast) {
  if (!sim || !state_dev) return fail(CF_E_ARG, "NULL argument");
  if (!sim->have_state) return fail(CF_E_STATE, "cf_set_state needs a prior cf_reset (world parameters)");
  sim->md_valid = false; sim->cost_valid = false; sim->rearmed = true;
  if (broadcast) {
    CF_CUDA(cudaMemcpyAsync(sim->bcast_buf, state_dev, sizeof(float) * sim->D, cudaMemcpyDeviceToDevice, sim->stream));
    sim->pending_bcast = true;
    return CF_OK;
  }
  sim->pending_bcast = false;
  return launch_set_state(sim, state_dev, 0);
}

extern "C" int cf_set_plan_state(cf_sim *sim, const float *eps_dev, const float *cost_run_dev) {
  if (!sim) return fail(CF_E_ARG, "sim is NULL");
  { int rc = materialise(sim); if (rc != CF_OK) return rc; }
  const size_t MN = (size_t)sim->MN;
  if (eps_dev) {
    if (!sim->eps) return fail(CF_E_ARG, "no AR(1) noise state: needs CF_CMD_NOMINAL_PLUS_NOISE with noise_beta != 0");
    CF_CUDA(cudaMemcpyAsync(sim->eps, eps_dev, sizeof(float) * 4 * MN, cudaMemcpyDeviceToDevice, sim->stream));
  }
  if (cost_run_dev) {
    if (!sim->cost_run) return fail(CF_E_ARG, "cost_on is 0");
    CF_CUDA(cudaMemcpyAsync(sim->cost_run, cost_run_dev, sizeof(float) * MN, cudaMemcpyDeviceToDevice, sim->stream));
  }
  sim->cost_valid = false; sim->rearmed = false;
  return CF_OK;
}

extern "C" int cf_set_full(cf_sim *sim, const float *state_dev, const float *ctrl_dev, const float *wparam_dev,
                           const float *min_d2_dev, int64_t step_counter) {
  if (!sim) return fail(CF_E_ARG, "sim is NULL");
  if (step_counter >= ((int64_t)1 << 32)) return fail(CF_E_SHAPE, "step_counter must be < 2^32");
  { int rc = materialise(sim); if (rc != CF_OK) return rc; }
  sim->md_valid = false; sim->cost_valid = false; sim->rearmed = false;
  const size_t MN = (size_t)sim->MN;
  if (state_dev) CF_CUDA(cudaMemcpyAsync(sim->state, state_dev, sizeof(float) * sim->D * MN, cudaMemcpyDeviceToDevice, sim->stream));
  if (ctrl_dev) CF_CUDA(cudaMemcpyAsync(sim->ctrl, ctrl_dev, sizeof(float) * kCtrlPlanes * MN, cudaMemcpyDeviceToDevice, sim->stream));
  if (wparam_dev) {
    CF_CUDA(cudaMemcpyAsync(sim->wparam, wparam_dev, sizeof(float) * sim->P * (size_t)sim->M, cudaMemcpyDeviceToDevice, sim->stream));
    sim->opt |= OPT_RANDP;     // the planes are now authoritative
    sim->wparam_foreign = true; // ... and the create-time bounds on the coefficients no longer hold
  }
  if (min_d2_dev) {
    if (!sim->min_d2) return fail(CF_E_ARG, "no obstacles configured");
    CF_CUDA(cudaMemcpyAsync(sim->min_d2, min_d2_dev, sizeof(float) * kMaxObst * MN, cudaMemcpyDeviceToDevice, sim->stream));
  }
  if (step_counter >= 0) {
    set_counters_kernel<<<1, 1, 0, sim->stream>>>(sim->counters, (uint32_t)step_counter, 0);
    CF_CUDA(cudaGetLastError());
    sim->s_host = step_counter;
  }
  sim->have_state = true;
  return CF_OK;
}

// Checkpoint restore of what cf_set_full leaves out: the tick / record counters and the record-slot table.
extern "C" int cf_set_counters(cf_sim *sim, const uint32_t counters_host[4], const uint32_t *rec_table_dev) {
  if (!sim || !counters_host) return fail(CF_E_ARG, "NULL argument");
  if (!sim->have_state) return fail(CF_E_STATE, "cf_set_counters before cf_reset");
  set_counters4_kernel<<<1, 1, 0, sim->stream>>>(sim->counters, counters_host[0], counters_host[1], counters_host[2],
                                                 counters_host[3]);
  CF_CUDA(cudaGetLastError());
  if (rec_table_dev)
    CF_CUDA(cudaMemcpyAsync(sim->rec_table, rec_table_dev, sizeof(uint32_t) * kRecTableCap, cudaMemcpyDeviceToDevice, sim->stream));
  sim->s_host = counters_host[0];
  sim->n_rec_host = counters_host[3];
  return CF_OK;
}

// The record buffer of one cf_step call as a 2-D tensor for the TMA unit: [n_rec * D rows][MN columns] float32, box = 32
// columns x D rows (one warp's snapshot), no swizzle, no interleave.  cuTensorMapEncodeTiled is a driver-API entry
// point, fetched through the runtime so that the library links against libcudart only.  false = not available (the
// caller falls back to one 4-byte store per component).
typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                  const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
static EncodeTiledFn encode_tiled_fn() {
  static EncodeTiledFn fn = []() -> EncodeTiledFn {
    void *p = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) != cudaSuccess ||
        q != cudaDriverEntryPointSuccess) {
      (void)cudaGetLastError();
      return nullptr;
    }
    return (EncodeTiledFn)p;
  }();
  return fn;
}
static bool encode_record_map(CUtensorMap *map, float *record_dev, long long MN, long long n_rec, int D, int group) {
  EncodeTiledFn enc = encode_tiled_fn();
  if (!enc) return false;
  const cuuint64_t dims[2] = { (cuuint64_t)MN, (cuuint64_t)(n_rec * D) };
  const cuuint64_t strides[1] = { (cuuint64_t)MN * sizeof(float) };      // bytes, a multiple of 16 (MN % 32 == 0)
  const cuuint32_t box[2] = { 32u, (cuuint32_t)(D * group) }, elem[2] = { 1u, 1u };
  return enc(map, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, record_dev, dims, strides, box, elem, CU_TENSOR_MAP_INTERLEAVE_NONE,
             CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

// launch geometry.  One wave always suffices for the paper's sizes up to ~600k drones (64 warps/SM x 148 SMs), so the
// block size only decides how evenly the warps spread over the SMs: the fewer warps per SM, the smaller the block.
// SM count of the current device, asked once (148 on a B200; the same value if the query fails, e.g. without a device)
static long long sm_count() {
  static const long long n = []() -> long long {
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess ||
        sms < 1) {
      (void)cudaGetLastError();
      return 148;
    }
    return sms;
  }();
  return n;
}
static int pick_block(long long MN) {
  const long long sms = sm_count(), warps = (MN + 31) / 32;
  if (warps <= sms * 16) return 32;
  if (warps <= sms * 32) return 64;
  return kMaxBlock;
}
// Record-every-step runs (lean kernels): the largest block (<= 512 threads) that leaves the busiest scheduler with no
// more warps than one-warp blocks would.  The record tensor is [n_rec * D][MN]: a warp writes 128 bytes of each of D rows
// that lie MN * 4 bytes apart, and what HBM sustains for that pattern grows with the span one SM writes at a time --
// measured with a write-only kernel of the same pattern (profiles/r2_record_pattern.md): 4.75 TB/s at 32 threads per
// block, 5.0 at 128, 5.4 at 256, 6.1 - 6.7 at 512 (a linear fill: 6.9).
static int pick_block_rec(long long MN) {
  const long long sms = sm_count(), warps = (MN + 31) / 32;
  auto busiest = [&](long long b) {            // warps on the busiest scheduler with blocks of b warps
    const long long blocks = (warps + b - 1) / b, per_sm = (blocks + sms - 1) / sms;
    return (per_sm * b + 3) / 4;
  };
  int best = 1;
  for (int b = 2; b <= kMaxBlockRec / 32; b *= 2)
    if (busiest(b) <= busiest(1)) best = b;
  return 32 * best;
}

// Option bits of the instantiation that this simulator's configuration dispatches to in record mode rec_mode (-1: none).
// A request without any fidelity extra still lands on the general OPT_ALL / REC_RUNTIME kernel when no lean instantiation
// was built for it (e.g. the rotor or position interface of the first-principles model, RK4 on the abstracted model):
// everything that depends on WHICH kernel runs -- block size, snapshots per store, the pair-written record modes -- is
// decided from this, not from the request.
// Measurement switch: with CF_FORCE_GENERAL=1 in the environment when the simulator is created, every cf_step runs the
// general OPT_ALL kernel (which gates each feature at run time from the same parameters) even where a lean instantiation
// exists -- for like-for-like lean / general timings (bench.py).  Results agree to rounding.
static int dispatch_opt_bits(const cf_sim *sim) { return sim->opt | (sim->force_general ? OPT_EXTRAS : 0); }
static int dispatched_opt(const cf_sim *sim, int rec_mode) {
  int opt_used = 0;
  const bool found = sim->model == CF_MODEL_FIRST_PRINCIPLES
      ? launch_fp(sim->p.integrator, sim->p.iface, dispatch_opt_bits(sim), rec_mode, nullptr, nullptr, nullptr, nullptr, &opt_used, true)
      : launch_ab(sim->p.integrator, sim->p.iface, dispatch_opt_bits(sim), rec_mode, nullptr, nullptr, nullptr, nullptr, &opt_used, true);
  return found ? opt_used : -1;
}
static bool dispatches_lean(const cf_sim *sim, int rec_mode) {
  const int o = dispatched_opt(sim, rec_mode);
  return o >= 0 && !(o & OPT_EXTRAS);
}

static int do_launch(cf_sim *sim, const StepArgs *A, bool dry, const char **name, int *grid, int *block) {
  LaunchCfg L;
  const int rec_mode = A ? A->rec_mode : sim->last_rec_mode;    // a dry run describes the kernel of the last cf_step
  // the kernel stages the parameter rows whenever ITS compile-time options carry OPT_RANDP and N > 1, and the
  // dispatcher may pick a superset instantiation: size the staging area from the instantiation, not from the request
  const int opt_used = dispatched_opt(sim, rec_mode);
  if (opt_used < 0) return fail(CF_E_UNSUPPORTED, "no kernel instantiation for this configuration");
  const bool general = (opt_used & OPT_EXTRAS) != 0;            // the OPT_ALL kernel: launch bound kMaxBlock
  if (A) sim->last_rec_mode = A->rec_mode;
  if (A) sim->last_rec_heavy = (A->rec_mode == REC_TMA || A->rec_mode == REC_PAIR || A->rec_mode == REC_TMA_P) && A->record_every <= 4 && !general;
  L.block = sim->last_rec_heavy ? pick_block_rec(sim->MN) : pick_block(sim->MN);
  if (general && L.block > kMaxBlock) L.block = kMaxBlock;
  L.grid = grid_for(A ? A->i_end - A->i_begin : sim->MN, L.block);
  size_t smem_wp = ((opt_used & OPT_RANDP) && sim->N > 1) ? sizeof(float) * sim->P * (size_t)L.block : 0;
  size_t smem_rec = (A && (A->rec_mode == REC_TMA || A->rec_mode == REC_PAIR || A->rec_mode == REC_TMA_P)) ? kRecBufs * A->rec_group * sizeof(float) * sim->D * 32 * (size_t)(L.block / 32) : 0;
  L.smem = smem_wp > smem_rec ? smem_wp : smem_rec;
  L.stream = sim->stream;
  if (grid) *grid = L.grid;
  if (block) *block = L.block;
  bool ok = sim->model == CF_MODEL_FIRST_PRINCIPLES
      ? launch_fp(sim->p.integrator, sim->p.iface, dispatch_opt_bits(sim), rec_mode, A, &sim->dp, &L, name, nullptr, dry)
      : launch_ab(sim->p.integrator, sim->p.iface, dispatch_opt_bits(sim), rec_mode, A, &sim->dp, &L, name, nullptr, dry);
  if (!ok) return fail(CF_E_UNSUPPORTED, "no kernel instantiation for this configuration");
  return CF_OK;
}

extern "C" int cf_describe_launch(const cf_sim *sim, char *buf, size_t buf_len, int *grid, int *block) {
  if (!sim) return fail(CF_E_ARG, "sim is NULL");
  const char *name = "";
  int rc = do_launch(const_cast<cf_sim *>(sim), nullptr, true, &name, grid, block);
  if (rc != CF_OK) return rc;
  if (buf && buf_len) snprintf(buf, buf_len, "%s", name);
  return CF_OK;
}

// One cf_step call.  n_slices == 1: one launch over all drones.  n_slices > 1 (cf_rollout_host): consecutive launches over
// slices of `slice` drones on the simulator's stream -- every slice reads the same counters, the last one advances them --
// with after_slice(k, i0, i1) called after each launch (the caller queues that slice's result copy on another stream).
typedef int (*SliceFn)(void *ctx, int k, long long i0, long long i1);
static int step_launch(cf_sim *sim, const void *cmds_dev, int n_cmds, int cmd_hold, int n_steps, int record_every,
                       float *record_dev, size_t record_bytes, long long slice, SliceFn after_slice, void *ctx) {
  if (!sim || !cmds_dev) return fail(CF_E_ARG, "NULL argument");
  if (n_steps < 1 || cmd_hold < 1 || n_cmds < 1 || record_every < 0) return fail(CF_E_ARG, "n_steps, cmd_hold, n_cmds >= 1; record_every >= 0");
  if (!sim->have_state) return fail(CF_E_STATE, "cf_step before cf_reset");
  if ((long long)n_cmds * cmd_hold < n_steps) return fail(CF_E_SHAPE, "n_cmds * cmd_hold < n_steps");
  if (((uintptr_t)cmds_dev & 15) != 0) return fail(CF_E_BUFFER, "cmds must be 16-byte aligned");
  long long s0 = sim->s_host, n_rec = 0;
  if (s0 + n_steps >= ((long long)1 << 32)) return fail(CF_E_SHAPE, "step counter would overflow 32 bits");
  if (record_every > 0) {
    n_rec = (s0 + n_steps) / record_every - s0 / record_every;
    if (n_rec > 0 && (!record_dev || record_bytes < (size_t)n_rec * sim->D * (size_t)sim->MN * sizeof(float)))
      return fail(CF_E_BUFFER, "record buffer too small for %lld records", n_rec);
  }
  // The pair-written kernels (REC_PAIR, REC_*_P) have "attitude tick in the first step of each pair" compiled in, which
  // holds because THIS call starts at an even step (s0 below, the host mirror).  A launch captured into a CUDA graph is
  // replayed from whatever the DEVICE counter holds then -- odd, if the graph's total length is odd -- so a call made
  // during stream capture never takes a pair-written kernel: the run-time-scheduled ones are correct from any step.
  bool capturing = false;
  {
    cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
    if (cudaStreamIsCapturing(sim->stream, &cs) == cudaSuccess) capturing = cs != cudaStreamCaptureStatusNone;
    else (void)cudaGetLastError();
  }
  StepArgs A;
  A.state = sim->state; A.ctrl = sim->ctrl; A.wparam = sim->wparam; A.min_d2 = sim->min_d2;
  A.bcast = sim->pending_bcast ? sim->bcast_buf : nullptr; A.md_drone = sim->md_drone;
  A.eps = sim->eps; A.cost_run = sim->cost_run; A.cost_drone = sim->cost_drone;
  A.worlds_per_ctrl = sim->p.worlds_per_ctrl; A.n_cmds = n_cmds;
  A.counters = sim->counters; A.rec_table = sim->rec_table;
  A.cmds = (const float4 *)cmds_dev; A.record = record_dev;
  A.MN = sim->MN; A.M = sim->M; A.N = sim->N; A.world_offset = sim->p.world_offset;
  A.n_steps = n_steps; A.cmd_hold = cmd_hold; A.record_every = record_every; A.n_rec_cap = (int)n_rec;
  memset(&A.rec_map, 0, sizeof(A.rec_map));
  A.rec_mode = n_rec > 0 ? REC_SCALAR : REC_NONE;
  memset(&A.rec_map1, 0, sizeof(A.rec_map1));
  A.rec_group = 1;
  if (n_rec > 0 && sim->MN % 32 == 0 && ((uintptr_t)record_dev & 15) == 0) {
    // snapshots per bulk-tensor store: worth it only when records are frequent; bounded by the shared memory the
    // resident warps can have (two tiles of rec_group * D * 128 bytes per warp; <= 48 KB per block, <= 200 KB per SM with
    // at most 20 resident warps, the lean kernels' launch bound) and by the number of records of this call
    int group = 1;
    const bool lean_tma = dispatches_lean(sim, REC_TMA);        // grouped stores and the large blocks are the lean kernels'
    if (record_every <= 4 && lean_tma) {
      const int block = pick_block_rec(sim->MN);
      const long long warps = (sim->MN + 31) / 32, bw = block / 32, blocks = (warps + bw - 1) / bw;
      long long resident = ((blocks + sm_count() - 1) / sm_count()) * bw;    // warps on the busiest SM
      if (resident > 20) resident = 20;
      const size_t tile = sizeof(float) * sim->D * 32;
      for (int g = kRecGroupMax; g > 1 && group == 1; --g)
        if (g <= n_rec && kRecBufs * g * tile * (size_t)resident <= 200 * 1024) group = g;
    }
    // the pair schedule as a compile-time fact (REC_PAIR): every step recorded, two snapshots per store, attitude tick
    // every second step starting with this call's first, an even number of steps in command runs of even length
    const bool pair = !capturing && group >= 2 && record_every == 1 && sim->model == CF_MODEL_FIRST_PRINCIPLES &&
        sim->p.iface == CF_IF_ATTITUDE && sim->p.integrator == CF_RK4 && dispatches_lean(sim, REC_PAIR) && sim->dp.att_div == 2 &&
        s0 % 2 == 0 && n_steps % 2 == 0 && cmd_hold != 1 && (cmd_hold % 2 == 0 || cmd_hold >= n_steps) && n_rec == n_steps;
    if (pair) group = 2;
    if (encode_record_map(&A.rec_map, record_dev, sim->MN, n_rec, sim->D, group) &&
        (group == 1 || encode_record_map(&A.rec_map1, record_dev, sim->MN, n_rec, sim->D, 1))) {
      if (group == 1) A.rec_map1 = A.rec_map;
      A.rec_mode = REC_TMA;
      A.rec_group = group;
      if (pair) A.rec_mode = REC_PAIR;
    }
  }
  // pair-written loops for the other record modes (REC_*_P, cf_device.cuh): nominal-plant first-principles kernels with
  // the attitude interface, tick period 2, an even number of steps from an even step in command runs of even length,
  // records never, every step, or with an even period
  if (!capturing && A.rec_mode != REC_PAIR && sim->model == CF_MODEL_FIRST_PRINCIPLES && sim->p.iface == CF_IF_ATTITUDE &&
      (sim->opt & ~OPT_RANDP) == 0 && sim->dp.att_div == 2 && s0 % 2 == 0 && n_steps % 2 == 0 && cmd_hold != 1 &&
      (cmd_hold % 2 == 0 || cmd_hold >= n_steps) && (record_every <= 1 || record_every % 2 == 0) &&
      dispatches_lean(sim, A.rec_mode + REC_NONE_P))     // (a parameter-randomised plant has no _P instantiation: it runs
    A.rec_mode += REC_NONE_P;        // REC_NONE / REC_SCALAR / REC_TMA -> their _P forms   the general kernel, base modes only)
  A.seed_lo = (uint32_t)(sim->seed & 0xFFFFFFFFu); A.seed_hi = (uint32_t)(sim->seed >> 32);
  for (int r = 0; r < 10; ++r) {      // Philox key schedule: k += (0x9E3779B9, 0xBB67AE85) per round
    A.rk[2 * r] = A.seed_lo + (uint32_t)r * 0x9E3779B9u;
    A.rk[2 * r + 1] = A.seed_hi + (uint32_t)r * 0xBB67AE85u;
  }
  if (slice <= 0 || slice >= sim->MN) slice = sim->MN;
  bool launched = false;
  for (long long i0 = 0, k = 0; i0 < sim->MN; i0 += slice, ++k) {
    A.i_begin = (int)i0;
    A.i_end = (int)(i0 + slice < sim->MN ? i0 + slice : sim->MN);
    A.advance = A.i_end == sim->MN;
    A.ang_bound_ok = sim->wparam_foreign ? 0 : 1;
    int rc = do_launch(sim, &A, false, nullptr, nullptr, nullptr);
    if (rc == CF_OK) {
      const cudaError_t e = cudaGetLastError();
      if (e != cudaSuccess) rc = fail(CF_E_CUDA, "rollout kernel launch: %s", cudaGetErrorString(e));
    }
    if (rc == CF_OK) {
      launched = true;
      if (after_slice) rc = after_slice(ctx, (int)k, A.i_begin, A.i_end);
    }
    if (rc != CF_OK) {
      // earlier slices have advanced their drones (and consumed a pending broadcast) while the counters have not moved:
      // the planes are a mixture of two steps.  The simulator refuses to continue from them (cf.h: cf_rollout_host).
      if (launched) sim->have_state = false;
      return rc;
    }
  }
  sim->s_host = s0 + n_steps;
  sim->n_rec_host += n_rec;
  sim->pending_bcast = false;
  sim->md_valid = sim->min_d2 != nullptr;
  sim->cost_valid = sim->cost_run != nullptr;
  sim->last_fresh = sim->rearmed; sim->last_s0 = s0; sim->last_n_steps = n_steps; sim->last_n_cmds = n_cmds;
  sim->last_cmd_hold = cmd_hold; sim->rearmed = false;
  return CF_OK;
}

extern "C" int cf_step(cf_sim *sim, const void *cmds_dev, int n_cmds, int cmd_hold, int n_steps, int record_every,
                       float *record_dev, size_t record_bytes) {
  return step_launch(sim, cmds_dev, n_cmds, cmd_hold, n_steps, record_every, record_dev, record_bytes, 0, nullptr, nullptr);
}

// ---------------------------------------------------------------------------------------------------------------
// host-buffer (end-to-end) path
static size_t cmd_bytes(const cf_sim *sim, int n_cmds) {
  size_t per = sim->p.cmd_source == CF_CMD_NOMINAL_PLUS_NOISE ? (size_t)sim->p.n_ctrl : (size_t)sim->MN;
  return align256(sizeof(float) * 4 * per * (size_t)n_cmds);
}
static long long n_records(const cf_sim *sim, int n_steps, int record_every) {
  if (record_every <= 0) return 0;
  return (sim->s_host + n_steps) / record_every - sim->s_host / record_every;
}

extern "C" size_t cf_staging_bytes(const cf_sim *sim, int n_cmds, int n_steps, int record_every) {
  if (!sim || n_cmds < 1 || n_steps < 1) return 0;
  return cmd_bytes(sim, n_cmds) + align256((size_t)n_records(sim, n_steps, record_every) * sim->D * (size_t)sim->MN * sizeof(float));
}

extern "C" int cf_step_host(cf_sim *sim, const void *cmds_host, int n_cmds, int cmd_hold, int n_steps, int record_every,
                            float *record_host, size_t record_bytes, void *staging_dev, size_t staging_bytes) {
  if (!sim || !cmds_host || !staging_dev) return fail(CF_E_ARG, "NULL argument");
  if (n_cmds < 1 || n_steps < 1) return fail(CF_E_ARG, "n_cmds, n_steps >= 1");
  if (((uintptr_t)staging_dev & 255) != 0) return fail(CF_E_BUFFER, "staging must be 256-byte aligned");
  size_t need = cf_staging_bytes(sim, n_cmds, n_steps, record_every);
  if (staging_bytes < need) return fail(CF_E_BUFFER, "staging too small: %zu < %zu", staging_bytes, need);
  size_t cb = cmd_bytes(sim, n_cmds);
  size_t rb = (size_t)n_records(sim, n_steps, record_every) * sim->D * (size_t)sim->MN * sizeof(float);
  if (rb > 0 && (!record_host || record_bytes < rb)) return fail(CF_E_BUFFER, "host record buffer too small");
  size_t per = sim->p.cmd_source == CF_CMD_NOMINAL_PLUS_NOISE ? (size_t)sim->p.n_ctrl : (size_t)sim->MN;
  CF_CUDA(cudaMemcpyAsync(staging_dev, cmds_host, sizeof(float) * 4 * per * (size_t)n_cmds, cudaMemcpyHostToDevice, sim->stream));
  float *rec_dev = (float *)((char *)staging_dev + cb);
  int rc = cf_step(sim, staging_dev, n_cmds, cmd_hold, n_steps, record_every, rec_dev, rb);
  if (rc != CF_OK) return rc;
  if (rb > 0) CF_CUDA(cudaMemcpyAsync(record_host, rec_dev, rb, cudaMemcpyDeviceToHost, sim->stream));
  CF_CUDA(cudaStreamSynchronize(sim->stream));
  return CF_OK;
}

// One fused rollout driven from HOST buffers with the result copies overlapped (the planning shape of configs[2]):
// the drones are advanced in n_slices consecutive launches on the simulator's stream; after each launch an event is
// recorded and a second stream copies that slice of the final state planes (a 2-D copy: D rows of `slice` floats, pitch
// MN floats) and of the per-drone minimum distance to the host while the next slice computes.
struct RolloutCopy { cf_sim *sim; float *state_host, *md_host; };
static int rollout_copy_slice(void *ctx, int k, long long i0, long long i1) {
  RolloutCopy *c = (RolloutCopy *)ctx;
  cf_sim *sim = c->sim;
  cudaEvent_t ev = sim->slice_ev[k];
  CF_CUDA(cudaEventRecord(ev, sim->stream));
  CF_CUDA(cudaStreamWaitEvent(sim->copy_stream, ev, 0));
  const size_t pitch = sizeof(float) * (size_t)sim->MN, width = sizeof(float) * (size_t)(i1 - i0);
  CF_CUDA(cudaMemcpy2DAsync(c->state_host + i0, pitch, sim->state + i0, pitch, width, (size_t)sim->D, cudaMemcpyDeviceToHost,
                            sim->copy_stream));
  if (c->md_host)
    CF_CUDA(cudaMemcpyAsync(c->md_host + i0, sim->md_drone + i0, width, cudaMemcpyDeviceToHost, sim->copy_stream));
  return CF_OK;
}
extern "C" int cf_rollout_host(cf_sim *sim, const float *x0_host, const void *cmds_host, int n_cmds, int cmd_hold,
                               int n_steps, float *state_host, float *min_dist_host, void *staging_dev,
                               size_t staging_bytes, int n_slices) {
  if (!sim || !cmds_host || !state_host || !staging_dev) return fail(CF_E_ARG, "NULL argument");
  if (n_cmds < 1 || n_steps < 1) return fail(CF_E_ARG, "n_cmds, n_steps >= 1");
  if (n_slices < 1 || n_slices > 16) return fail(CF_E_ARG, "n_slices in 1..16");
  if (!sim->have_state) return fail(CF_E_STATE, "cf_rollout_host before cf_reset");
  if (min_dist_host && (!sim->min_d2 || sim->N != 1))
    return fail(CF_E_UNSUPPORTED, "min_dist_host needs obstacles and one drone per world (the rollout epilogue's per-drone read-out)");
  if (((uintptr_t)staging_dev & 255) != 0) return fail(CF_E_BUFFER, "staging must be 256-byte aligned");
  const size_t cb = cmd_bytes(sim, n_cmds), xb = align256(sizeof(float) * sim->D);
  if (staging_bytes < cb + xb) return fail(CF_E_BUFFER, "staging too small: %zu < %zu", staging_bytes, cb + xb);
  if (!sim->copy_stream) {
    CF_CUDA(cudaStreamCreateWithFlags(&sim->copy_stream, cudaStreamNonBlocking));
    sim->copy_stream_owned = true;
  }
  for (int k = 0; k < n_slices; ++k)
    if (!sim->slice_ev[k]) CF_CUDA(cudaEventCreateWithFlags(&sim->slice_ev[k], cudaEventDisableTiming));
  const size_t per = sim->p.cmd_source == CF_CMD_NOMINAL_PLUS_NOISE ? (size_t)sim->p.n_ctrl : (size_t)sim->MN;
  CF_CUDA(cudaMemcpyAsync(staging_dev, cmds_host, sizeof(float) * 4 * per * (size_t)n_cmds, cudaMemcpyHostToDevice, sim->stream));
  if (x0_host) {                         // every drone starts from this state (lazy broadcast, folded into the launches)
    float *x0_dev = (float *)((char *)staging_dev + cb);
    CF_CUDA(cudaMemcpyAsync(x0_dev, x0_host, sizeof(float) * sim->D, cudaMemcpyHostToDevice, sim->stream));
    int rc = cf_set_state(sim, x0_dev, 1);
    if (rc != CF_OK) return rc;
  }
  // slices of whole blocks (1024 drones is a multiple of every block size the launcher picks)
  long long slice = ((sim->MN + n_slices - 1) / n_slices + 1023) / 1024 * 1024;
  RolloutCopy ctx = { sim, state_host, min_dist_host };
  int rc = step_launch(sim, staging_dev, n_cmds, cmd_hold, n_steps, 0, nullptr, 0, slice, rollout_copy_slice, &ctx);
  // both streams are drained whatever happened: copies of the slices that did run may still be in flight
  cudaError_t e1 = cudaStreamSynchronize(sim->copy_stream), e2 = cudaStreamSynchronize(sim->stream);
  if (rc != CF_OK) return rc;
  CF_CUDA(e1);
  CF_CUDA(e2);
  return CF_OK;
}

extern "C" int cf_get_state(cf_sim *sim, float *out_dev) {
  if (!sim || !out_dev) return fail(CF_E_ARG, "NULL argument");
  { int rc = materialise(sim); if (rc != CF_OK) return rc; }
  CF_CUDA(cudaMemcpyAsync(out_dev, sim->state, sizeof(float) * sim->D * (size_t)sim->MN, cudaMemcpyDeviceToDevice, sim->stream));
  return CF_OK;
}
extern "C" int cf_get_state_host(cf_sim *sim, float *out_host) {
  if (!sim || !out_host) return fail(CF_E_ARG, "NULL argument");
  { int rc = materialise(sim); if (rc != CF_OK) return rc; }
  CF_CUDA(cudaMemcpyAsync(out_host, sim->state, sizeof(float) * sim->D * (size_t)sim->MN, cudaMemcpyDeviceToHost, sim->stream));
  CF_CUDA(cudaStreamSynchronize(sim->stream));
  return CF_OK;
}

// make cost_drone hold J of the current planes (it already does straight after a cf_step: rollout epilogue)
int cf_refresh_cost(cf_sim *sim) {
  if (!sim->cost_run) return fail(CF_E_ARG, "cost_on is 0");
  { int rc = materialise(sim); if (rc != CF_OK) return rc; }
  if (!sim->cost_valid) {
    cost_readout_kernel<<<grid_for(sim->MN, 256), 256, 0, sim->stream>>>(sim->state, sim->min_d2, sim->cost_run,
                                                                          sim->cost_drone, sim->MN, sim->dp);
    CF_CUDA(cudaGetLastError());
    sim->cost_valid = true;
  }
  return CF_OK;
}

static int aux_source(cf_sim *sim, int which, const void **src, size_t *bytes) {
  const size_t MN = (size_t)sim->MN;
  { int rc = materialise(sim); if (rc != CF_OK) return rc; }
  switch (which) {
    case CF_AUX_COUNTERS: *src = sim->counters; *bytes = 4 * sizeof(uint32_t); return CF_OK;
    case CF_AUX_CTRL: *src = sim->ctrl; *bytes = sizeof(float) * kCtrlPlanes * MN; return CF_OK;
    case CF_AUX_WORLD_PARAMS: *src = sim->wparam; *bytes = sizeof(float) * sim->P * (size_t)sim->M; return CF_OK;
    case CF_AUX_REC_TABLE: *src = sim->rec_table; *bytes = sizeof(uint32_t) * kRecTableCap; return CF_OK;
    case CF_AUX_MIN_D2:
      if (!sim->min_d2) return fail(CF_E_ARG, "no obstacles configured");
      *src = sim->min_d2; *bytes = sizeof(float) * kMaxObst * MN; return CF_OK;
    case CF_AUX_EPS:
      if (!sim->eps) return fail(CF_E_ARG, "no AR(1) noise state: needs CF_CMD_NOMINAL_PLUS_NOISE with noise_beta != 0");
      *src = sim->eps; *bytes = sizeof(float) * 4 * MN; return CF_OK;
    case CF_AUX_COST_RUN:
      if (!sim->cost_run) return fail(CF_E_ARG, "cost_on is 0");
      *src = sim->cost_run; *bytes = sizeof(float) * MN; return CF_OK;
    case CF_AUX_COST: {
      int rc = cf_refresh_cost(sim);
      if (rc != CF_OK) return rc;
      *src = sim->cost_drone; *bytes = sizeof(float) * MN; return CF_OK;
    }
  }
  return fail(CF_E_ARG, "bad aux selector %d", which);
}

static int launch_min_dist(cf_sim *sim, float *out_dev) {
  if (!sim->min_d2) return fail(CF_E_ARG, "no obstacles configured");
  { int rc = materialise(sim); if (rc != CF_OK) return rc; }
  if (sim->md_valid && sim->N == 1) {   // the rollout kernel's epilogue already reduced obstacles and steps per drone
    CF_CUDA(cudaMemcpyAsync(out_dev, sim->md_drone, sizeof(float) * (size_t)sim->M, cudaMemcpyDeviceToDevice, sim->stream));
    return CF_OK;
  }
  if (sim->N < 8) {
    min_dist_small_n_kernel<<<grid_for(sim->M, 256), 256, 0, sim->stream>>>(sim->min_d2, out_dev, sim->M, sim->N, sim->MN, sim->dp);
  } else {
    long long threads = sim->M * 32;
    min_dist_kernel<<<grid_for(threads, 128), 128, 0, sim->stream>>>(sim->min_d2, out_dev, sim->M, sim->N, sim->MN, sim->dp);
  }
  CF_CUDA(cudaGetLastError());
  return CF_OK;
}

static int launch_nonfinite(cf_sim *sim, uint32_t *out_dev) {
  { int rc = materialise(sim); if (rc != CF_OK) return rc; }
  nonfinite_init_kernel<<<1, 1, 0, sim->stream>>>(out_dev);
  nonfinite_kernel<<<grid_for(sim->MN, 256), 256, 0, sim->stream>>>(sim->state, sim->D, sim->MN, out_dev);
  CF_CUDA(cudaGetLastError());
  return CF_OK;
}

extern "C" int cf_get_aux(cf_sim *sim, int which, void *out_dev) {
  if (!sim || !out_dev) return fail(CF_E_ARG, "NULL argument");
  if (which == CF_AUX_MIN_DIST) return launch_min_dist(sim, (float *)out_dev);
  if (which == CF_AUX_NONFINITE) return launch_nonfinite(sim, (uint32_t *)out_dev);
  const void *src; size_t bytes;
  int rc = aux_source(sim, which, &src, &bytes);
  if (rc != CF_OK) return rc;
  CF_CUDA(cudaMemcpyAsync(out_dev, src, bytes, cudaMemcpyDeviceToDevice, sim->stream));
  return CF_OK;
}

extern "C" int cf_get_aux_host(cf_sim *sim, int which, void *out_host, void *scratch_dev, size_t scratch_bytes) {
  if (!sim || !out_host) return fail(CF_E_ARG, "NULL argument");
  const void *src; size_t bytes;
  if (which == CF_AUX_MIN_DIST) {
    bytes = sizeof(float) * (size_t)sim->M;
    if (!scratch_dev || scratch_bytes < bytes) return fail(CF_E_BUFFER, "scratch_dev must hold M floats");
    int rc = launch_min_dist(sim, (float *)scratch_dev);
    if (rc != CF_OK) return rc;
    src = scratch_dev;
  } else if (which == CF_AUX_NONFINITE) {
    bytes = 2 * sizeof(uint32_t);
    if (!scratch_dev || scratch_bytes < bytes || ((uintptr_t)scratch_dev & 3)) return fail(CF_E_BUFFER, "scratch_dev must hold 2 uint32");
    int rc = launch_nonfinite(sim, (uint32_t *)scratch_dev);
    if (rc != CF_OK) return rc;
    src = scratch_dev;
  } else {
    int rc = aux_source(sim, which, &src, &bytes);
    if (rc != CF_OK) return rc;
  }
  CF_CUDA(cudaMemcpyAsync(out_host, src, bytes, cudaMemcpyDeviceToHost, sim->stream));
  CF_CUDA(cudaStreamSynchronize(sim->stream));
  return CF_OK;
}

extern "C" int64_t cf_step_counter(const cf_sim *sim) { return sim ? sim->s_host : -1; }

extern "C" int cf_sync_counters(cf_sim *sim) {
  if (!sim) return fail(CF_E_ARG, "sim is NULL");
  uint32_t c[4];
  CF_CUDA(cudaMemcpyAsync(c, sim->counters, sizeof(c), cudaMemcpyDeviceToHost, sim->stream));
  CF_CUDA(cudaStreamSynchronize(sim->stream));
  sim->s_host = c[0];
  sim->n_rec_host = c[3];
  return CF_OK;
}

extern "C" int cf_debug_philox(uint64_t seed, const uint32_t ctr[4], uint32_t out[4]) {
  if (!ctr || !out) return fail(CF_E_ARG, "NULL argument");
  philox4x32_10((uint32_t)(seed & 0xFFFFFFFFu), (uint32_t)(seed >> 32), ctr[0], ctr[1], ctr[2], ctr[3], out);
  return CF_OK;
}

extern "C" int cf_debug_philox_dev(cf_sim *sim, uint64_t seed, const uint32_t *ctr_dev, int n, uint32_t *words_dev,
                                   float *uniform_dev, float *normal_dev) {
  if (!sim || !ctr_dev || n < 1) return fail(CF_E_ARG, "bad argument");
  philox_debug_kernel<<<grid_for(n, 128), 128, 0, sim->stream>>>((uint32_t)(seed & 0xFFFFFFFFu), (uint32_t)(seed >> 32),
                                                                 ctr_dev, n, words_dev, uniform_dev, normal_dev);
  CF_CUDA(cudaGetLastError());
  return CF_OK;
}
