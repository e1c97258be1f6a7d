// cf_device.cuh -- device side of libcf.so: the fused rollout kernel (thread = drone, state in registers across all
// sub-steps) and its building blocks.  float32 arithmetic, uint32 counters / Philox.  sm_100a only.
//
// What each piece computes is defined by PAPER.md Eqs. (1)-(10) and the readings in DESIGN.md; citations are at
// each function.  This file shares nothing with oracle/ (the float64 CPU oracle).
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace cf {

constexpr int kMaxObst = 8;
constexpr int kCtrlPlanes = 14;
constexpr int kRecTableCap = 4096;
constexpr int kRecGroupMax = 4;   // snapshots per bulk-tensor store, at most
constexpr int kRecBufs = 2;       // record staging tiles per warp (TMA path: one in flight, one being filled; 3 and 4
                                  // measured no faster)

// option bits of a kernel instantiation
enum : int {
  OPT_RANDP = 1,    // plant parameters come from the per-world planes (domain randomisation)
  OPT_DIST = 2,     // per-step Philox force disturbance
  OPT_OBST = 4,     // running minimum squared distance to the obstacle spheres
  OPT_NOISE = 8,    // command = clip(nominal[k] + sigma * z), z from Philox (CF_CMD_NOMINAL_PLUS_NOISE)
  OPT_EXTRAS = 16,  // full Eq. (6) (asymmetric + quadratic), thrust/torque polynomials, Eq. (5) gyro, body drag,
                    // simplified AB variant
  OPT_COST = 32,    // rollout cost for the sampling-based planner (reading R27)
  OPT_AR = 64,      // OPT_NOISE with temporally correlated noise (AR(1), reading R25): eps kept as simulator state
  OPT_ALL = 127
};
enum : int { MODEL_FP = 0, MODEL_AB = 1 };
enum : int { INTEG_EULER = 0, INTEG_RK4 = 1 };
enum : int { IF_ROTOR = 0, IF_TORQUE = 1, IF_ATTITUDE = 2, IF_POSITION = 3 };
enum : int { STREAM_INIT = 0, STREAM_PARAM = 1, STREAM_DIST = 2, STREAM_NOISE = 3 };

struct Counters {          // device-resident, 64 B
  uint32_t s, att_ticks, pos_ticks, n_rec_total;
  uint32_t blocks_done, pad[11];
};

// Uniform (per-launch) constants; lives in the kernel parameter constant bank.
struct DevParams {
  float h, half_h, h_sixth, h_att, h_pos, g;
  // nominal plant
  float mass, inv_mass, J[3], inv_J[3], lever, kf[3], km[3];
  float cv_up, cv_dn, cd_up, cd_dn, Jp_rad /* Jp * 2pi/60 */, Ca[3];
  float ab_a[3], ab_b[3], ab_c[3], ab_ctau, ab_cf;
  int   ab_thrust_dyn, thrust_poly /* kf0 or kf1 != 0 */, has_drag, has_gyro;
  // controller (nominal parameters, reading R11)
  float inv_4lever, inv_4kappa, f_rotor_max, inv_kf2, rpm_min, rpm_max, thrust_min, thrust_max, tilt_max;
  float kR[3], kW[3], kI[3], iR_max, Jnom[3];
  float kp[3], kd[3], ki[3], ip_max[3];
  float dist_sigma;
  int   use_noise;   // cmd_source == CF_CMD_NOMINAL_PLUS_NOISE
  int   n_obst;
  float obst[kMaxObst][4];        // cx cy cz r (read-out)
  float4 obst_q[kMaxObst];        // (-2cx, -2cy, -2cz, c.c): d^2 = |p|^2 + q.(p,1); unused slots (0,0,0,+inf)
  float obst_x[kMaxObst], obst_y[kMaxObst], obst_z[kMaxObst];   // the same -2c components as three constant-bank rows
  float noise_sigma[4], cmd_lo[4], cmd_hi[4];
  float noise_beta, noise_gain;    // R25: AR(1) coefficient and sqrt(1 - beta^2)
  float cost_goal[3], cost_hw_pos, cost_hw_vel;   // R27: h w_pos, h w_vel (running), and the read-out terms:
  float cost_w_term, cost_w_obs, cost_d_safe, cost_w_coll;
  int   cost_on;
  int   att_div, pos_div;
  float hover_thrust, hover_rpm;   // reading R20: held commands after a reset / set_state
  // abstracted model, bound on the growth of the Euler angles (lean Euler step): over ALL worlds of this simulator
  // max_j |h a_j| and max_j |1 + h b_j| (nominal coefficients x randomisation ranges); see run_angles_bounded
  float bnd_ha, bnd_hb1;
};

struct StepArgs {
  float *state;            // [D][MN]
  float *ctrl;             // [14][MN]
  const float *wparam;     // [P][M]
  float *min_d2;           // [8][MN] or nullptr
  const float *bcast;      // [D] or nullptr: start every drone from this state with re-armed controllers (lazy cf_set_state)
  float *md_drone;         // [MN] or nullptr: per-drone min over obstacles and steps of |p - c_j| - r_j (epilogue)
  float *eps;              // [4][MN] or nullptr: AR(1) command-noise state (kept when noise_beta != 0)
  float *cost_run;         // [MN] or nullptr: running rollout cost
  float *cost_drone;       // [MN] or nullptr: total rollout cost J (epilogue, R27)
  long long worlds_per_ctrl;   // R26: nominal sequence of a world = cmds + (local world / worlds_per_ctrl) * n_cmds
  int n_cmds;
  Counters *counters;
  uint32_t *rec_table;     // [kRecTableCap]
  const float4 *cmds;      // [K][MN] or [K]
  float *record;           // [n_rec][D][MN]
  long long MN, M, N, world_offset;
  int n_steps, cmd_hold, record_every, n_rec_cap;
  int rec_mode;            // REC_NONE / REC_SCALAR (one 4-byte store per component) / REC_TMA (bulk-tensor store of a
                           // [D][32] shared-memory tile; needs MN % 32 == 0 and a 16-byte aligned record buffer)
  uint32_t seed_lo, seed_hi;
  uint32_t rk[20];         // Philox round keys (k0_r, k1_r), r = 0..9, precomputed on the host from the seed
  int rec_group;           // REC_TMA: snapshots per bulk-tensor store (1..kRecGroupMax), chosen by the host from the
                           // record period and the shared memory the resident warps can have
  alignas(64) CUtensorMap rec_map;    // REC_TMA: the record buffer as the 2-D tensor [n_rec * D][MN], box = 32 x rec_group * D
  alignas(64) CUtensorMap rec_map1;   // the same tensor with box = 32 x D (partial last group)
  // (appended: the offsets of everything above -- the Philox keys are read with 8 / 16-byte constant loads -- stay put)
  int i_begin, i_end;         // (M N < 2^31) this launch advances the drones [i_begin, i_end) (a slice of the batch: cf_rollout_host; else [0, MN))
  int advance;                // this launch advances the device-side counters (the last slice of a call)
  int ang_bound_ok;           // DevParams.bnd_* hold for every world (false after cf_set_full replaced the parameter planes)
};

// ---------------------------------------------------------------------------------------------------------------
// Philox4x32-10 (Salmon et al. 2011), reading C9: key = (seed lo, seed hi), counter = (world, drone, index, stream)
__host__ __device__ __forceinline__ void philox4x32_10(uint32_t k0, uint32_t k1, uint32_t c0, uint32_t c1,
                                                       uint32_t c2, uint32_t c3, uint32_t out[4]) {
#pragma unroll
  for (int r = 0; r < 10; ++r) {
#ifdef __CUDA_ARCH__
    uint32_t hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
    uint32_t hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
#else
    uint64_t p0 = (uint64_t)0xD2511F53u * c0, p1 = (uint64_t)0xCD9E8D57u * c2;
    uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0, hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
#endif
    uint32_t n0 = hi1 ^ c1 ^ k0, n2 = hi0 ^ c3 ^ k1;
    c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
    k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// ---------------------------------------------------------------------------------------------------------------
// Special-function unit (MUFU) approximations.  The rollout loop is instruction-issue bound (profiles/), so the
// transcendental work goes to the otherwise idle XU pipe instead of ~30-instruction FMA-pipe software routines.
// Error budget: sin/cos.approx abs err <= 2^-20.9 on [-2pi, 2pi],
// lg2.approx abs err <= 2^-22 on the logarithm, sqrt.approx <= 2 ulp -- all >= 2 orders below the 1e-4 per-step bar.
__device__ __forceinline__ float mufu_sin(float x) { float y; asm("sin.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float mufu_cos(float x) { float y; asm("cos.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float mufu_lg2(float x) { float y; asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float mufu_sqrt(float x) { float y; asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }

// sin / cos of a physical angle inside the step loop.  |x| <= 2 pi: MUFU; beyond (never in the paper's workloads,
// attitude commands are clipped to +-pi) the accurate library routine, so the result is defined for any input.
__device__ __forceinline__ void sincos_step(float x, float *s, float *c) {
  if (fabsf(x) <= 6.2831853f) { *s = mufu_sin(x); *c = mufu_cos(x); }
  else sincosf(x, s, c);
}

// the same 10 rounds with the key schedule precomputed (uniform per launch): 2 IMAD.WIDE + 2 LOP3 per round
__device__ __forceinline__ void philox4x32_10_rk(const uint32_t (&rk)[20], uint32_t c0, uint32_t c1, uint32_t c2,
                                                 uint32_t c3, uint32_t out[4]) {
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    uint32_t hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
    uint32_t hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
    uint32_t n0 = hi1 ^ c1 ^ rk[2 * r], n2 = hi0 ^ c3 ^ rk[2 * r + 1];
    c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// atan2 / asin for the position controller: odd minimax polynomial of degree 15 on [0,1] (fitted for this build, max
// abs error 1.3e-7 evaluated in float32) after the usual octant reduction; one MUFU.RCP instead of a division.
__device__ __forceinline__ float fast_atan2f(float y, float x) {
  float ax = fabsf(x), ay = fabsf(y);
  float mx = fmaxf(fmaxf(ax, ay), 1e-30f), mn = fminf(ax, ay);
  float a = __fdividef(mn, mx), t = a * a;
  float p = -0.004054096061736345f;
  p = fmaf(p, t, 0.021861093118786812f);
  p = fmaf(p, t, -0.05590933561325073f);
  p = fmaf(p, t, 0.09641948342323303f);
  p = fmaf(p, t, -0.13908515870571136f);
  p = fmaf(p, t, 0.19946537911891937f);
  p = fmaf(p, t, -0.33329856395721436f);
  p = fmaf(p, t, 0.9999993443489075f);
  float r = p * a;
  r = ay > ax ? 1.57079632679f - r : r;
  r = x < 0.0f ? 3.14159265359f - r : r;
  return copysignf(r, y);
}
__device__ __forceinline__ float fast_asinf(float x) {       // |x| <= 1
  return fast_atan2f(x, mufu_sqrt(fmaxf(fmaf(-x, x, 1.0f), 0.0f)));
}

// the three Euler angles at once: one range check for all
__device__ __forceinline__ void sincos3_step(const float *a, float *s, float *c) {
  if (fmaxf(fmaxf(fabsf(a[0]), fabsf(a[1])), fabsf(a[2])) <= 6.2831853f) {
#pragma unroll
    for (int j = 0; j < 3; ++j) { s[j] = mufu_sin(a[j]); c[j] = mufu_cos(a[j]); }
  } else {
#pragma unroll
    for (int j = 0; j < 3; ++j) sincosf(a[j], &s[j], &c[j]);
  }
}

// The same for ANY angle without a branch: r = a - 2 pi k, k = rint(a / 2 pi) by magic-number rounding (exact for
// |a / 2 pi| < 2^22), 2 pi split in two float32 constants (Cody-Waite: 2 pi = 6.2831855 - 1.7484556e-7), so |r| <= pi
// whatever a is, then MUFU.  For |a| < pi: k = 0 and r = a exactly.  Four FMA-pipe instructions per angle more than the
// tested form above -- but a step loop that uses it has no branch diamond left, and the compiler then schedules across
// the step boundary and keeps loop constants live.  Used by the per-step-command (flat) loop of the lean abstracted-model
// kernels, where that is worth 7 % (configs[2]: 0.699 -> 0.653 ms); the held-command loops measured no gain (planner
// rollout -0.5 %, configs[3] -8 %) and keep the tested form.
__device__ __forceinline__ float reduce_to_pi(float a) {
  const float k = fmaf(a, 0.15915494309f, 12582912.0f) - 12582912.0f;
  return fmaf(k, 1.7484556e-7f, fmaf(k, -6.2831855f, a));
}
__device__ __forceinline__ void sincos3_any(const float *a, float *s, float *c) {
#pragma unroll
  for (int j = 0; j < 3; ++j) { const float r = reduce_to_pi(a[j]); s[j] = mufu_sin(r); c[j] = mufu_cos(r); }
}

// reading R18: 23-bit midpoint uniform in (0,1), exact in float32:  u = ((x >> 9) + 0.5) 2^-23.
// Built as the float 1.m (m = x >> 9) minus (1 - 2^-24): both are multiples of 2^-24, the difference is exact.
__device__ __forceinline__ float u01(uint32_t x) {
  return __uint_as_float(0x3F800000u | (x >> 9)) - 0.99999994f;
}
// 2 pi (u - 1/2): 1.m - 1.5 is exact (a multiple of 2^-23 in [-1/2, 1/2)); the half-ulp offset 2^-24 enters through
// the FMA's addend.  The Box-Muller angle is thus taken on (-pi, pi), where MUFU sin/cos are accurate.
__device__ __forceinline__ float angle_centered(uint32_t x) {
  float t = __uint_as_float(0x3F800000u | (x >> 9)) - 1.5f;
  return fmaf(t, 6.28318530718f, 6.28318530718f * 5.9604644775390625e-8f);
}

// Box-Muller (C9): r = sqrt(-2 ln ua), (z0, z1) = r (cos 2 pi ub, sin 2 pi ub).
// cos(2 pi ub) = -cos(2 pi (ub - 1/2)) and likewise for sin, so the sign goes into r.
__device__ __forceinline__ void normal_pair(uint32_t xa, uint32_t xb, float &z0, float &z1) {
  float ua = u01(xa);
  float ang = angle_centered(xb);
  float r = -mufu_sqrt(-1.38629436112f * mufu_lg2(ua));     // -2 ln u = -2 ln2 * lg2 u
  z0 = r * mufu_cos(ang); z1 = r * mufu_sin(ang);
}

__device__ __forceinline__ float clipf(float v, float lo, float hi) { return fminf(fmaxf(v, lo), hi); }

// ---------------------------------------------------------------------------------------------------------------
// Plant parameters of one world, in the derived form the derivative wants.
template <int MODEL, int OPT> struct Plant;

template <int OPT> struct Plant<MODEL_FP, OPT> {
  float inv_m, inv_J[3], cJ[3];      // cJ = ((Jy-Jz)/Jx, (Jz-Jx)/Jy, (Jx-Jy)/Jz): Euler's equation cross term
  float kf2, km2, cv;                // lean rotor / thrust model
  float kfm2, ct[3];                 // lean: 2 kf2/m ; (l kf2/Jx, l kf2/Jy, km2/Jz)
  float rc2, rc3, rc4, rho4, rho1;   // lean: closed-form first-order rotor lag inside RK4 / Euler, z = h cv (see integrate_fp_lean)
  float J[3], kf0, kf1, km0, km1, cv_dn, cd_up, cd_dn;   // only read when OPT_EXTRAS

  __device__ __forceinline__ void set(const DevParams &P, float m, float Jx, float Jy, float Jz, const float kf[3],
                                      const float km[3], float cvu, float cvd, float cdu, float cdd) {
    inv_m = 1.0f / m;
    inv_J[0] = 1.0f / Jx; inv_J[1] = 1.0f / Jy; inv_J[2] = 1.0f / Jz;
    cJ[0] = (Jy - Jz) * inv_J[0]; cJ[1] = (Jz - Jx) * inv_J[1]; cJ[2] = (Jx - Jy) * inv_J[2];
    kf2 = kf[2]; km2 = km[2]; cv = cvu;
    kfm2 = 2.0f * kf2 * inv_m;
    ct[0] = P.lever * kf2 * inv_J[0]; ct[1] = P.lever * kf2 * inv_J[1]; ct[2] = km2 * inv_J[2];
    const float z = P.h * cv;
    rc2 = 1.0f - 0.5f * z;
    rc3 = 1.0f - 0.5f * z * rc2;
    rc4 = 1.0f - z * rc3;
    rho4 = 1.0f - z * (1.0f - z * (0.5f - z * (1.0f / 6.0f - z * (1.0f / 24.0f))));
    rho1 = 1.0f - z;
    J[0] = Jx; J[1] = Jy; J[2] = Jz;
    kf0 = kf[0]; kf1 = kf[1]; km0 = km[0]; km1 = km[1]; cv_dn = cvd; cd_up = cdu; cd_dn = cdd;
  }
  __device__ __forceinline__ void load(const DevParams &P, const float *wp, long long M, long long w, bool randp) {
    if (randp) {
      float kf[3] = { wp[4 * M + w], wp[5 * M + w], wp[6 * M + w] };
      float km[3] = { wp[7 * M + w], wp[8 * M + w], wp[9 * M + w] };
      set(P, wp[w], wp[M + w], wp[2 * M + w], wp[3 * M + w], kf, km, wp[10 * M + w], wp[11 * M + w], wp[12 * M + w],
          wp[13 * M + w]);
    } else {
      set(P, P.mass, P.J[0], P.J[1], P.J[2], P.kf, P.km, P.cv_up, P.cv_dn, P.cd_up, P.cd_dn);
    }
  }
};

template <int OPT> struct Plant<MODEL_AB, OPT> {
  float inv_m, a[3], b[3], c[3], ctau;
  // lean Euler step (integrate_ab_euler_lean): the step length folded into the coefficients
  float ha[3], hb1[3], hc[3], hct, omhct, h_cf_m;      // h a, 1 + h b, h c, h c_tau, 1 - h c_tau, h c_f / m
  __device__ __forceinline__ void fold_step(const DevParams &P) {
#pragma unroll
    for (int j = 0; j < 3; ++j) { ha[j] = P.h * a[j]; hb1[j] = fmaf(P.h, b[j], 1.0f); hc[j] = P.h * c[j]; }
    hct = P.h * ctau; omhct = 1.0f - hct; h_cf_m = P.h * P.ab_cf * inv_m;
  }
  __device__ __forceinline__ void load(const DevParams &P, const float *wp, long long M, long long w, bool randp) {
    load_raw(P, wp, M, w, randp);
    fold_step(P);
  }
  __device__ __forceinline__ void load_raw(const DevParams &P, const float *wp, long long M, long long w, bool randp) {
    if (randp) {
      inv_m = 1.0f / wp[w];
#pragma unroll
      for (int j = 0; j < 3; ++j) { a[j] = wp[(1 + j) * M + w]; b[j] = wp[(4 + j) * M + w]; c[j] = wp[(7 + j) * M + w]; }
      ctau = wp[10 * M + w];
    } else {
      inv_m = P.inv_mass;
#pragma unroll
      for (int j = 0; j < 3; ++j) { a[j] = P.ab_a[j]; b[j] = P.ab_b[j]; c[j] = P.ab_c[j]; }
      ctau = P.ab_ctau;
    }
  }
};

// rotation matrix of a scalar-last unit quaternion
__device__ __forceinline__ void quat_to_R(const float *q, float R[3][3]) {
  float x = q[0], y = q[1], z = q[2], w = q[3];
  float xx = x * x, yy = y * y, zz = z * z, xy = x * y, xz = x * z, yz = y * z, wx = w * x, wy = w * y, wz = w * z;
  R[0][0] = 1.0f - 2.0f * (yy + zz); R[0][1] = 2.0f * (xy - wz);        R[0][2] = 2.0f * (xz + wy);
  R[1][0] = 2.0f * (xy + wz);        R[1][1] = 1.0f - 2.0f * (xx + zz); R[1][2] = 2.0f * (yz - wx);
  R[2][0] = 2.0f * (xz - wy);        R[2][1] = 2.0f * (yz + wx);        R[2][2] = 1.0f - 2.0f * (xx + yy);
}
// reading R13: R = Rz(yaw) Ry(pitch) Rx(roll)
__device__ __forceinline__ void euler_to_R(float roll, float pitch, float yaw, float R[3][3]) {
  float sr, cr, sp, cp, sy, cy;
  sincosf(roll, &sr, &cr); sincosf(pitch, &sp, &cp); sincosf(yaw, &sy, &cy);
  R[0][0] = cy * cp; R[0][1] = cy * sp * sr - sy * cr; R[0][2] = cy * sp * cr + sy * sr;
  R[1][0] = sy * cp; R[1][1] = sy * sp * sr + cy * cr; R[1][2] = sy * sp * cr - cy * sr;
  R[2][0] = -sp;     R[2][1] = cp * sr;                R[2][2] = cp * cr;
}

// ---------------------------------------------------------------------------------------------------------------
// First-principles derivative, Eqs. (1)-(6) (C2).  x = p(0-2) q(3-6) v(7-9) w(10-12) Omega(13-16).
// Mixing matrix C1: sx = (-,-,+,+), sy = (-,+,+,-), sz = (-,+,-,+) (X configuration, spin +,-,+,-).
template <int OPT>
__device__ __forceinline__ void deriv_fp(const DevParams &P, const Plant<MODEL_FP, OPT> &pl, const float *x,
                                         const float *rpm_cmd, const float *fdist, float *dx) {
  const float *q = x + 3, *v = x + 7, *w = x + 10, *Om = x + 13;
  constexpr bool EX = (OPT & OPT_EXTRAS) != 0;
  float dOm[4];
  float F, tau[3];   // F [N] ; tau already divided by nothing (N m)
  if (!EX) {
    // Eq. (6) with c_v^ = c_v_, c_d = 0: first-order lag;  f = kf2 W^2, m = km2 W^2
    float w2[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) { dOm[k] = pl.cv * (rpm_cmd[k] - Om[k]); w2[k] = Om[k] * Om[k]; }
    float A = w2[0] + w2[1], B = w2[2] + w2[3], C = w2[1] + w2[2], D = w2[0] + w2[3];
    float E = w2[1] + w2[3], G = w2[0] + w2[2];
    F = pl.kf2 * (A + B);
    tau[0] = (P.lever * pl.kf2) * (B - A);
    tau[1] = (P.lever * pl.kf2) * (C - D);
    tau[2] = pl.km2 * (E - G);
  } else {
    float f[4], mk[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      float e = rpm_cmd[k] - Om[k];
      bool up = e >= 0.0f;
      float cv = up ? pl.cv : pl.cv_dn, cd = up ? pl.cd_up : pl.cd_dn;
      dOm[k] = cv * e + cd * (rpm_cmd[k] * rpm_cmd[k] - Om[k] * Om[k]);
      f[k] = pl.kf0 + Om[k] * (pl.kf1 + pl.kf2 * Om[k]);
      mk[k] = pl.km0 + Om[k] * (pl.km1 + pl.km2 * Om[k]);
    }
    F = (f[0] + f[1]) + (f[2] + f[3]);
    tau[0] = P.lever * ((f[2] + f[3]) - (f[0] + f[1]));
    tau[1] = P.lever * ((f[1] + f[2]) - (f[0] + f[3]));
    tau[2] = (mk[1] + mk[3]) - (mk[0] + mk[2]);
    if (P.has_gyro) {   // Eq. (5), reading R2: Jp (-wy S, +wx S, -dS), S = W1 - W2 + W3 - W4 in rad/s
      float S = (Om[0] - Om[1]) + (Om[2] - Om[3]), dS = (dOm[0] - dOm[1]) + (dOm[2] - dOm[3]);
      tau[0] -= P.Jp_rad * w[1] * S;
      tau[1] += P.Jp_rad * w[0] * S;
      tau[2] -= P.Jp_rad * dS;
    }
  }
  // Eq. (3): dv = z_B F/m + f_dist/m - g e_z (+ body drag)
  float zx = 2.0f * (q[0] * q[2] + q[3] * q[1]);
  float zy = 2.0f * (q[1] * q[2] - q[3] * q[0]);
  float zz = 1.0f - 2.0f * (q[0] * q[0] + q[1] * q[1]);
  float acc = F * pl.inv_m;
  float ax = zx * acc, ay = zy * acc, az = zz * acc - P.g;
  if (OPT & OPT_DIST) { ax += fdist[0] * pl.inv_m; ay += fdist[1] * pl.inv_m; az += fdist[2] * pl.inv_m; }
  if (EX && P.has_drag) {
    float R[3][3];
    quat_to_R(q, R);
    float fb[3];
#pragma unroll
    for (int j = 0; j < 3; ++j) fb[j] = P.Ca[j] * (R[0][j] * v[0] + R[1][j] * v[1] + R[2][j] * v[2]);
    ax += (R[0][0] * fb[0] + R[0][1] * fb[1] + R[0][2] * fb[2]) * pl.inv_m;
    ay += (R[1][0] * fb[0] + R[1][1] * fb[1] + R[1][2] * fb[2]) * pl.inv_m;
    az += (R[2][0] * fb[0] + R[2][1] * fb[1] + R[2][2] * fb[2]) * pl.inv_m;
  }
  dx[7] = ax; dx[8] = ay; dx[9] = az;
  // Eq. (4), diagonal J: dw = tau/J + cJ * (w_j w_k)
  dx[10] = tau[0] * pl.inv_J[0] + pl.cJ[0] * (w[1] * w[2]);
  dx[11] = tau[1] * pl.inv_J[1] + pl.cJ[1] * (w[2] * w[0]);
  dx[12] = tau[2] * pl.inv_J[2] + pl.cJ[2] * (w[0] * w[1]);
  // Eq. (2), reading R1: dq = 1/2 q (x) (w, 0)
  dx[3] = 0.5f * (q[3] * w[0] + q[1] * w[2] - q[2] * w[1]);
  dx[4] = 0.5f * (q[3] * w[1] + q[2] * w[0] - q[0] * w[2]);
  dx[5] = 0.5f * (q[3] * w[2] + q[0] * w[1] - q[1] * w[0]);
  dx[6] = -0.5f * (q[0] * w[0] + q[1] * w[1] + q[2] * w[2]);
  // Eq. (1)
  dx[0] = v[0]; dx[1] = v[1]; dx[2] = v[2];
#pragma unroll
  for (int k = 0; k < 4; ++k) dx[13 + k] = dOm[k];
}

// Abstracted derivative, Eqs. (7)-(10) (C3).  x = p(0-2) Psi(3-5) v(6-8) dPsi(9-11) f_Sigma(12); u = attitude cmd.
template <int OPT>
__device__ __forceinline__ void deriv_ab(const DevParams &P, const Plant<MODEL_AB, OPT> &pl, const float *x,
                                         const float *u, const float *fdist, float *dx) {
  constexpr bool EX = (OPT & OPT_EXTRAS) != 0;
  float sn[3], cs[3];
  sincos3_step(x + 3, sn, cs);
  const float sr = sn[0], cr = cs[0], sp = sn[1], cp = cs[1], sy = sn[2], cy = cs[2];
  float zx = cy * sp * cr + sy * sr, zy = sy * sp * cr - cy * sr, zz = cp * cr;
  float fS = (EX && !P.ab_thrust_dyn) ? u[3] : x[12];
  float acc = (P.ab_cf * fS) * pl.inv_m;
  float ax = zx * acc, ay = zy * acc, az = zz * acc - P.g;
  if (OPT & OPT_DIST) { ax += fdist[0] * pl.inv_m; ay += fdist[1] * pl.inv_m; az += fdist[2] * pl.inv_m; }
  if (EX && P.has_drag) {
    float R[3][3];
    R[0][0] = cy * cp; R[0][1] = cy * sp * sr - sy * cr; R[0][2] = zx;
    R[1][0] = sy * cp; R[1][1] = sy * sp * sr + cy * cr; R[1][2] = zy;
    R[2][0] = -sp;     R[2][1] = cp * sr;                R[2][2] = zz;
    const float *v = x + 6;
    float fb[3];
#pragma unroll
    for (int j = 0; j < 3; ++j) fb[j] = P.Ca[j] * (R[0][j] * v[0] + R[1][j] * v[1] + R[2][j] * v[2]);
    ax += (R[0][0] * fb[0] + R[0][1] * fb[1] + R[0][2] * fb[2]) * pl.inv_m;
    ay += (R[1][0] * fb[0] + R[1][1] * fb[1] + R[1][2] * fb[2]) * pl.inv_m;
    az += (R[2][0] * fb[0] + R[2][1] * fb[1] + R[2][2] * fb[2]) * pl.inv_m;
  }
  dx[0] = x[6]; dx[1] = x[7]; dx[2] = x[8];
  dx[6] = ax; dx[7] = ay; dx[8] = az;
#pragma unroll
  for (int j = 0; j < 3; ++j) {
    dx[3 + j] = x[9 + j];
    dx[9 + j] = pl.a[j] * x[3 + j] + pl.b[j] * x[9 + j] + pl.c[j] * u[j];
  }
  dx[12] = (EX && !P.ab_thrust_dyn) ? 0.0f : pl.ctau * (u[3] - x[12]);
}

template <int MODEL, int OPT>
__device__ __forceinline__ void deriv(const DevParams &P, const Plant<MODEL, OPT> &pl, const float *x,
                                      const float *u, const float *fdist, float *dx) {
  if constexpr (MODEL == MODEL_FP) deriv_fp<OPT>(P, pl, x, u, fdist, dx);
  else deriv_ab<OPT>(P, pl, x, u, fdist, dx);
}

// ---------------------------------------------------------------------------------------------------------------
// Lean first-principles step (no OPT_EXTRAS): Eqs. (1)-(4) + Eq. (6) with c_v^ = c_v_, c_d = 0 + pure-quadratic thrust
// and torque curves, the same C4 scheme as the generic integrator below, restated with fewer instructions:
//  * the rotor lag is linear and decoupled, so its RK4 stages and update are exact closed forms in z = h c_v
//    (SURVEY.md C12): with e = W - W_cmd, stage speeds are W_cmd + e (1, 1 - z/2, 1 - z/2 + z^2/4, 1 - z + z^2/2 - z^3/4)
//    and W+ = W_cmd + e (1 - z + z^2/2 - z^3/6 + z^4/24)   [Euler: W+ = W_cmd + e (1 - z)];
//  * dv does not depend on v or p, so p+ = p + h v + h^2/6 (a1 + a2 + a3) and no stage velocities are formed;
//  * rates carry their constant factors: a uses 2 k_f/m, dw uses l k_f/J, dq is 2 q-dot (stepped with h/2).
struct FpRates { float a[3], dw[3], dq[4]; };

template <int OPT>
__device__ __forceinline__ void fp_lean_rates(const Plant<MODEL_FP, OPT> &pl, const float *q, const float *w,
                                              const float *Om, const float *fa, FpRates &r) {
  float w2[4];
#pragma unroll
  for (int k = 0; k < 4; ++k) w2[k] = Om[k] * Om[k];
  float A = w2[0] + w2[1], B = w2[2] + w2[3], C = w2[1] + w2[2], Dd = w2[0] + w2[3];
  float E = w2[1] + w2[3], G = w2[0] + w2[2];
  float acc2 = pl.kfm2 * (A + B);                             // 2 F / m
  float zx = fmaf(q[0], q[2], q[3] * q[1]);                   // z_B = (2 zx, 2 zy, 1 - 2 zh)
  float zy = fmaf(q[1], q[2], -(q[3] * q[0]));
  float zh = fmaf(q[0], q[0], q[1] * q[1]);
  r.a[0] = fmaf(zx, acc2, fa[0]);
  r.a[1] = fmaf(zy, acc2, fa[1]);
  r.a[2] = fmaf(-zh, acc2, fmaf(0.5f, acc2, fa[2]));          // fa[2] already holds f_z/m - g
  r.dw[0] = fmaf(pl.cJ[0], w[1] * w[2], pl.ct[0] * (B - A));
  r.dw[1] = fmaf(pl.cJ[1], w[2] * w[0], pl.ct[1] * (C - Dd));
  r.dw[2] = fmaf(pl.cJ[2], w[0] * w[1], pl.ct[2] * (E - G));
  r.dq[0] = fmaf(q[3], w[0], fmaf(q[1], w[2], -(q[2] * w[1])));
  r.dq[1] = fmaf(q[3], w[1], fmaf(q[2], w[0], -(q[0] * w[2])));
  r.dq[2] = fmaf(q[3], w[2], fmaf(q[0], w[1], -(q[1] * w[0])));
  r.dq[3] = -fmaf(q[0], w[0], fmaf(q[1], w[1], q[2] * w[2]));
}

template <int INTEG, int OPT>
__device__ __forceinline__ void integrate_fp_lean(const DevParams &P, const Plant<MODEL_FP, OPT> &pl, float *x,
                                                  const float *rpm_cmd, const float *fdist) {
  float *p = x, *q = x + 3, *v = x + 7, *w = x + 10, *Om = x + 13;
  float fa[3] = { 0.0f, 0.0f, -P.g };
  if (OPT & OPT_DIST) { fa[0] = fdist[0] * pl.inv_m; fa[1] = fdist[1] * pl.inv_m; fa[2] = fmaf(fdist[2], pl.inv_m, -P.g); }
  float e[4];
#pragma unroll
  for (int k = 0; k < 4; ++k) e[k] = Om[k] - rpm_cmd[k];
  const float hq = 0.5f * P.h;                                // dq is twice the quaternion rate
  FpRates r1;
  fp_lean_rates<OPT>(pl, q, w, Om, fa, r1);
  if constexpr (INTEG == INTEG_EULER) {
#pragma unroll
    for (int j = 0; j < 3; ++j) { p[j] = fmaf(P.h, v[j], p[j]); v[j] = fmaf(P.h, r1.a[j], v[j]); w[j] = fmaf(P.h, r1.dw[j], w[j]); }
#pragma unroll
    for (int j = 0; j < 4; ++j) { q[j] = fmaf(hq, r1.dq[j], q[j]); Om[j] = fmaf(e[j], pl.rho1, rpm_cmd[j]); }
  } else {
    float qs[4], ws[3], Os[4];
    FpRates r2, r3, r4;
#pragma unroll
    for (int j = 0; j < 4; ++j) { qs[j] = fmaf(0.5f * hq, r1.dq[j], q[j]); Os[j] = fmaf(e[j], pl.rc2, rpm_cmd[j]); }
#pragma unroll
    for (int j = 0; j < 3; ++j) ws[j] = fmaf(P.half_h, r1.dw[j], w[j]);
    fp_lean_rates<OPT>(pl, qs, ws, Os, fa, r2);
#pragma unroll
    for (int j = 0; j < 4; ++j) { qs[j] = fmaf(0.5f * hq, r2.dq[j], q[j]); Os[j] = fmaf(e[j], pl.rc3, rpm_cmd[j]); }
#pragma unroll
    for (int j = 0; j < 3; ++j) ws[j] = fmaf(P.half_h, r2.dw[j], w[j]);
    fp_lean_rates<OPT>(pl, qs, ws, Os, fa, r3);
#pragma unroll
    for (int j = 0; j < 4; ++j) { qs[j] = fmaf(hq, r3.dq[j], q[j]); Os[j] = fmaf(e[j], pl.rc4, rpm_cmd[j]); }
#pragma unroll
    for (int j = 0; j < 3; ++j) ws[j] = fmaf(P.h, r3.dw[j], w[j]);
    fp_lean_rates<OPT>(pl, qs, ws, Os, fa, r4);
    const float h2_6 = P.h * P.h_sixth, hq6 = 0.5f * P.h_sixth;
#pragma unroll
    for (int j = 0; j < 3; ++j) {
      float a12 = r1.a[j] + r2.a[j];
      p[j] = fmaf(P.h, v[j], fmaf(h2_6, a12 + r3.a[j], p[j]));
      v[j] = fmaf(P.h_sixth, fmaf(2.0f, r3.a[j], a12 + r2.a[j]) + r4.a[j], v[j]);
      w[j] = fmaf(P.h_sixth, fmaf(2.0f, r3.dw[j], fmaf(2.0f, r2.dw[j], r1.dw[j])) + r4.dw[j], w[j]);
    }
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      q[j] = fmaf(hq6, fmaf(2.0f, r3.dq[j], fmaf(2.0f, r2.dq[j], r1.dq[j])) + r4.dq[j], q[j]);
      Om[j] = fmaf(e[j], pl.rho4, rpm_cmd[j]);
    }
  }
  float inv = rsqrtf(fmaf(q[0], q[0], fmaf(q[1], q[1], fmaf(q[2], q[2], q[3] * q[3]))));
#pragma unroll
  for (int j = 0; j < 4; ++j) q[j] *= inv;
}

// Lean abstracted-model Euler step (no OPT_EXTRAS): Eqs. (7)-(10) with x+ = x + h f(x) restated with the step length
// folded into per-world coefficients and the held command folded into `held` = (h c_j u_j, h c_tau u_3), which changes
// only when the command does:  Psi' += ...: dPsi+ = (1 + h b) dPsi + h a Psi + h c u  (2 FFMA per axis),
// f+ = (1 - h c_tau) f + h c_tau u_3 (1 FFMA), v+ = v + z_B (h c_f f / m) - h g e_z.  Same scheme as the generic
// integrator (algebraically identical restatements are free), ~10 instructions fewer per step.
template <int OPT>
__device__ __forceinline__ void integrate_ab_euler_lean(const DevParams &P, const Plant<MODEL_AB, OPT> &pl, float *x,
                                                        const float *held, const float *fdist, const float *sn,
                                                        const float *cs) {   // sn, cs: sin / cos of the pre-step Psi
  const float sr = sn[0], cr = cs[0], sp = sn[1], cp = cs[1], sy = sn[2], cy = cs[2];
  const float t = sp * cr;
  const float zx = fmaf(cy, t, sy * sr), zy = fmaf(sy, t, -(cy * sr)), zz = cp * cr;
  const float hacc = pl.h_cf_m * x[12];
#pragma unroll
  for (int j = 0; j < 3; ++j) {
    x[j] = fmaf(P.h, x[6 + j], x[j]);                                    // p += h v (old v)
    const float psi = x[3 + j];
    x[3 + j] = fmaf(P.h, x[9 + j], psi);                                 // Psi += h dPsi (old dPsi)
    x[9 + j] = fmaf(pl.ha[j], psi, fmaf(pl.hb1[j], x[9 + j], held[j]));  // Eq. (10)
  }
  x[6] = fmaf(zx, hacc, x[6]);
  x[7] = fmaf(zy, hacc, x[7]);
  x[8] = fmaf(zz, hacc, x[8] - P.h * P.g);
  if (OPT & OPT_DIST) {
    const float hm = P.h * pl.inv_m;
    x[6] = fmaf(hm, fdist[0], x[6]); x[7] = fmaf(hm, fdist[1], x[7]); x[8] = fmaf(hm, fdist[2], x[8]);
  }
  x[12] = fmaf(pl.omhct, x[12], held[3]);                                // Eq. (9)
}

// C4: explicit Euler / classical RK4, inputs held; q renormalised once per step, not inside the stages (R8-R10).
template <int MODEL, int INTEG, int OPT>
__device__ __forceinline__ void integrate(const DevParams &P, const Plant<MODEL, OPT> &pl, float *x, const float *u,
                                          const float *fdist, const float *held = nullptr, const float *sn = nullptr,
                                          const float *cs = nullptr) {
  constexpr int D = MODEL == MODEL_FP ? 17 : 13;
  if constexpr (MODEL == MODEL_AB && INTEG == INTEG_EULER && !(OPT & OPT_EXTRAS)) {
    integrate_ab_euler_lean<OPT>(P, pl, x, held, fdist, sn, cs);
    return;
  }
  if constexpr (MODEL == MODEL_FP && !(OPT & OPT_EXTRAS)) {
    integrate_fp_lean<INTEG, OPT>(P, pl, x, u, fdist);
    return;
  }
  float k[D];
  if constexpr (INTEG == INTEG_EULER) {
    deriv<MODEL, OPT>(P, pl, x, u, fdist, k);
#pragma unroll
    for (int j = 0; j < D; ++j) x[j] = fmaf(P.h, k[j], x[j]);
  } else {
    float xs[D], acc[D];
    deriv<MODEL, OPT>(P, pl, x, u, fdist, k);
#pragma unroll
    for (int j = 0; j < D; ++j) { acc[j] = k[j]; xs[j] = fmaf(P.half_h, k[j], x[j]); }
    deriv<MODEL, OPT>(P, pl, xs, u, fdist, k);
#pragma unroll
    for (int j = 0; j < D; ++j) { acc[j] = fmaf(2.0f, k[j], acc[j]); xs[j] = fmaf(P.half_h, k[j], x[j]); }
    deriv<MODEL, OPT>(P, pl, xs, u, fdist, k);
#pragma unroll
    for (int j = 0; j < D; ++j) { acc[j] = fmaf(2.0f, k[j], acc[j]); xs[j] = fmaf(P.h, k[j], x[j]); }
    deriv<MODEL, OPT>(P, pl, xs, u, fdist, k);
#pragma unroll
    for (int j = 0; j < D; ++j) x[j] = fmaf(P.h_sixth, acc[j] + k[j], x[j]);
  }
  if constexpr (MODEL == MODEL_FP) {
    float *q = x + 3;
    float inv = rsqrtf(q[0] * q[0] + q[1] * q[1] + q[2] * q[2] + q[3] * q[3]);
#pragma unroll
    for (int j = 0; j < 4; ++j) q[j] *= inv;
  } else if ((OPT & OPT_EXTRAS) && !P.ab_thrust_dyn) {
    x[12] = u[3];
  }
}

// ---------------------------------------------------------------------------------------------------------------
// C6 motor mixer (nominal parameters): (F_c, tau_des) -> rotor thrusts -> clip -> rpm -> clip
template <int OPT>
__device__ __forceinline__ void mixer(const DevParams &P, float Fc, const float *tau, float *rpm_cmd) {
  float a = 0.25f * Fc, bx = tau[0] * P.inv_4lever, by = tau[1] * P.inv_4lever, bz = tau[2] * P.inv_4kappa;
  float f[4] = { a - bx - by - bz, a - bx + by + bz, a + bx + by - bz, a + bx - by + bz };
#pragma unroll
  for (int k = 0; k < 4; ++k) {
    float fk = clipf(f[k], 0.0f, P.f_rotor_max);
    float r;
    if ((OPT & OPT_EXTRAS) && P.thrust_poly) {
      float disc = fmaxf(P.kf[1] * P.kf[1] - 4.0f * P.kf[2] * (P.kf[0] - fk), 0.0f);
      r = (sqrtf(disc) - P.kf[1]) * (0.5f * P.inv_kf2);
    } else {
      r = mufu_sqrt(fk * P.inv_kf2);
    }
    rpm_cmd[k] = clipf(r, P.rpm_min, P.rpm_max);
  }
}

// C5 attitude controller tick (reading R7).  Rd = columns of the desired rotation, hoisted to the command fetch.
template <int OPT>
__device__ __forceinline__ void attitude_tick(const DevParams &P, const float *q, const float *w, const float Rd[3][3],
                                              float Fc, float *iR, float *rpm_cmd) {
  float R[3][3];
  quat_to_R(q, R);
  // M = Rd^T R ; e_R = 1/2 (M32 - M23, M13 - M31, M21 - M12)
  auto Mij = [&](int i, int j) { return Rd[0][i] * R[0][j] + Rd[1][i] * R[1][j] + Rd[2][i] * R[2][j]; };
  float eR[3] = { 0.5f * (Mij(2, 1) - Mij(1, 2)), 0.5f * (Mij(0, 2) - Mij(2, 0)), 0.5f * (Mij(1, 0) - Mij(0, 1)) };
  float tau[3];
#pragma unroll
  for (int j = 0; j < 3; ++j) {
    iR[j] = clipf(fmaf(eR[j], P.h_att, iR[j]), -P.iR_max, P.iR_max);
    tau[j] = P.Jnom[j] * (-P.kR[j] * eR[j] - P.kW[j] * w[j] - P.kI[j] * iR[j]);
  }
  mixer<OPT>(P, Fc, tau, rpm_cmd);
}

// C7 geometric position controller tick (reading R16): target (x,y,z,yaw) -> attitude command (roll,pitch,yaw,F)
__device__ __forceinline__ void position_tick(const DevParams &P, const float *pos, const float *vel, const float *zB,
                                              const float *target, float *ip, float *att_cmd) {
  float t[3];
#pragma unroll
  for (int j = 0; j < 3; ++j) {
    float ep = target[j] - pos[j];
    ip[j] = clipf(fmaf(ep, P.h_pos, ip[j]), -P.ip_max[j], P.ip_max[j]);
    float ad = P.kp[j] * ep - P.kd[j] * vel[j] + P.ki[j] * ip[j] + (j == 2 ? P.g : 0.0f);
    t[j] = P.mass * ad;
  }
  float Fc = clipf(t[0] * zB[0] + t[1] * zB[1] + t[2] * zB[2], P.thrust_min, P.thrust_max);
  float inv = rsqrtf(fmaxf(t[0] * t[0] + t[1] * t[1] + t[2] * t[2], 1e-12f));     // 1 / max(|t|, 1e-6)
  float zd[3] = { t[0] * inv, t[1] * inv, t[2] * inv };
  float sy, cy;
  sincos_step(target[3], &sy, &cy);
  // y_d = z_d x x_c,  x_c = (cos yaw, sin yaw, 0)
  float yd[3] = { -zd[2] * sy, zd[2] * cy, zd[0] * sy - zd[1] * cy };
  float invy = rsqrtf(fmaxf(yd[0] * yd[0] + yd[1] * yd[1] + yd[2] * yd[2], 1e-12f));
  yd[0] *= invy; yd[1] *= invy; yd[2] *= invy;
  // x_d = y_d x z_d
  float xd[3] = { yd[1] * zd[2] - yd[2] * zd[1], yd[2] * zd[0] - yd[0] * zd[2], yd[0] * zd[1] - yd[1] * zd[0] };
  att_cmd[0] = clipf(fast_atan2f(yd[2], zd[2]), -P.tilt_max, P.tilt_max);
  att_cmd[1] = clipf(fast_asinf(clipf(-xd[2], -1.0f, 1.0f)), -P.tilt_max, P.tilt_max);
  att_cmd[2] = fast_atan2f(xd[1], xd[0]);
  att_cmd[3] = Fc;
}

// ---------------------------------------------------------------------------------------------------------------
// Record stream through the TMA unit (cp.async.bulk.tensor, SASS UTMASTG): the caller's record buffer is the 2-D tensor
// [n_rec * D rows][MN columns]; a warp parks its snapshot as a [D][32] tile in shared memory and ONE elected lane hands
// the whole tile to the copy engine.  The tile is double-buffered: the warp goes on computing while the engine drains.
__device__ __forceinline__ void fence_proxy_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void tma_store_tile_2d(const void *tmap, uint32_t smem_addr, int col, int row, int pred) {
  asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
               "@p cp.async.bulk.tensor.2d.global.shared::cta.bulk_group [%0, {%1, %2}], [%3];\n\t"
               "@p cp.async.bulk.commit_group;\n\t}"
               :: "l"(tmap), "r"(col), "r"(row), "r"(smem_addr), "r"(pred) : "memory");
}
template <int N> __device__ __forceinline__ void tma_store_wait_read() {
  asm volatile("cp.async.bulk.wait_group.read %0;" :: "n"(N) : "memory");
}

struct NoSmem { static constexpr bool value = false; };
struct InSmem { static constexpr bool value = true; };
template <int V> struct IntC { static constexpr int value = V; };
enum : int { REC_NONE = 0, REC_SCALAR = 1, REC_TMA = 2, REC_PAIR = 3, REC_NONE_P = 4, REC_SCALAR_P = 5, REC_TMA_P = 6,
             REC_RUNTIME = -1 };
// REC_PAIR: REC_TMA for the record-EVERY-step runs of the first-principles attitude-interface kernels (configs[4]), with
// the step loop written as pairs of steps whose schedule is a compile-time fact -- the attitude tick (period 2) in the
// first step, one bulk-tensor store of both snapshots after the second -- so the loop body has no branch at all.  The
// host selects it when record_every == 1, att_div == 2, two snapshots per store, and the call starts on an even step
// and runs an even number of steps in runs of even length (cf_api.cu); otherwise REC_TMA.
// REC_NONE_P / REC_SCALAR_P / REC_TMA_P: the same pair-written loop (tick in the first step of a pair as a compile-time
// fact) for the other record modes, with the record test BETWEEN steps / pairs (record_every 0, 1 or even): what the
// small batches gain -- one warp per scheduler, where every branch of the step is latency on the critical path
// (4096 worlds, RK4, every step recorded: 0.520 -> 0.444 us per step with the pair form).

// The rollout kernel.  One thread = one drone; the state, controller state, held commands and plant parameters stay
// in registers for all n_steps; HBM is touched for command loads, recorded states and the final store only.
//
// Lean instantiations (no OPT_EXTRAS) take their compiled-in options as unconditionally ON (the dispatcher hands them
// only requests with exactly those options; OPT_RANDP alone may be a superset, the parameter planes always hold valid
// values) and exist once per record mode REC (separate kernels: each gets its own register allocation), so the step
// loop carries no run-time feature test.  General instantiations (OPT_ALL, REC_RUNTIME) gate everything at run time.
// Launch bounds (measured on B200, profiles/r2_launch_config.md): blocks of at most 128 threads; abstracted-model lean
// kernels at >= 5 blocks / SM (<= 96 registers, 20 warps: best of 3..6 blocks and 64 / 128 / 256 threads on configs[2],
// configs[3] and the planner); first-principles lean kernels at >= 4 blocks (<= 128 registers, so that the 2048
// one-warp blocks of configs[4] are all resident: at > 146 registers they spill into a second wave, +50 % time).
constexpr int kMaxBlock = 128;
// The lean kernels' bounds are written as ONE block of 640 / 512 threads: the same register caps (<= 96 / <= 128), and
// blocks of up to 512 threads may be launched -- used when every step is recorded (see pick_block in cf_api.cu).
constexpr int kMaxBlockRec = 512;
// The position-interface abstracted-model kernels (configs[3]: no obstacle table, no Philox) need fewer registers and
// gain from a sixth resident block: bound 768 = 6 x 128 threads (<= 80 registers, 24 warps / SM): 5.98 -> 5.82 ms on
// configs[3]; the same bound costs the planning kernels (configs[2], planner) 10 % (measured sweep of bounds 576 .. 832).
constexpr int kBoundAbPos = 768;
template <int MODEL, int INTEG, int IFACE, int OPT, int REC>
__global__ void __launch_bounds__((OPT & OPT_EXTRAS) ? kMaxBlock : (MODEL == MODEL_AB ? (IFACE == IF_POSITION ? kBoundAbPos : 640) : 512), 1)
rollout_kernel(const __grid_constant__ StepArgs A, const __grid_constant__ DevParams P) {
  constexpr int D = MODEL == MODEL_FP ? 17 : 13;
  constexpr int NP = MODEL == MODEL_FP ? 14 : 11;
  constexpr bool FP = MODEL == MODEL_FP;
  constexpr bool GEN = (OPT & OPT_EXTRAS) != 0;
  constexpr bool HAS_ATT = FP && IFACE >= IF_ATTITUDE;       // attitude controller + mixer active
  constexpr bool HAS_POS = IFACE == IF_POSITION;
  extern __shared__ __align__(128) float wp_s[];             // [NP][span] per-world parameters of this block (N > 1);
                                                             // afterwards [warps][2][D][32] record staging tiles

  // obstacle table in shared memory for the held-command loop: one LDS.128 per sphere and step instead of two LDC.64
  // (sm_100a takes no constant-bank operands in FFMA, and the uniform registers are taken by the Philox keys and command
  // limits): mppi rollout 692 -> 653 us.  The flat per-step-command loop (configs[2]) is 7 % SLOWER with it (measured)
  // and keeps reading the table from the constant bank.
  __shared__ float4 obst_s[kMaxObst];
  if ((OPT & OPT_OBST) && threadIdx.x < kMaxObst) obst_s[threadIdx.x] = P.obst_q[threadIdx.x];
  if (OPT & OPT_OBST) __syncthreads();

  const long long MN = A.MN;
  // slices of the batch (cf_rollout_host) exist only for launches that record nothing: the recording lean kernels keep
  // the whole-batch geometry as a compile-time fact
  constexpr bool PAIRED = REC >= REC_PAIR;            // the step loop is written in pairs of steps
  constexpr int RECB = REC == REC_NONE_P ? REC_NONE : REC == REC_SCALAR_P ? REC_SCALAR : REC == REC_TMA_P ? REC_TMA : REC;   // record path
  constexpr bool SLICED = RECB == REC_NONE || REC == REC_RUNTIME;
  static_assert(!PAIRED || (MODEL == MODEL_FP && IFACE == IF_ATTITUDE), "pair-written loops: first-principles kernels, attitude interface");
  const int blk0 = (SLICED ? A.i_begin : 0) + (int)(blockIdx.x * blockDim.x);      // first drone of this block
  const int i_end = SLICED ? A.i_end : (int)MN;
  const long long i = blk0 + (int)threadIdx.x;
  const bool active = i < i_end;
  // the warp index as a value the compiler can prove warp-uniform (the TMA instruction takes uniform operands)
  const int warp_u = __shfl_sync(0xffffffffu, (int)(threadIdx.x >> 5), 0);
  // the device-side counters, broadcast from lane 0 so that the compiler can prove them (and every phase counter, loop
  // bound and record slot derived from them) warp-uniform: the step loop's control then runs on the uniform datapath
  // and the TMA store gets its operands without a per-lane uniformisation loop
  const uint32_t s0 = __shfl_sync(0xffffffffu, *((volatile uint32_t *)&A.counters->s), 0);
  const uint32_t rec0 = __shfl_sync(0xffffffffu, *((volatile uint32_t *)&A.counters->n_rec_total), 0);

  Plant<MODEL, OPT> pl;
  long long w = 0, n = 0;
  if (active) { w = i / A.N; n = i - w * A.N; }
  if ((OPT & OPT_RANDP) && A.N > 1) {
    // stage the parameter rows of the worlds this block touches in shared memory, then read them from there
    long long first = blk0;
    long long last = first + blockDim.x - 1 < i_end - 1 ? first + blockDim.x - 1 : i_end - 1;
    long long w_first = first / A.N;
    int span = (int)(last / A.N - w_first) + 1;
    for (int idx = threadIdx.x; idx < NP * span; idx += blockDim.x) {
      int pidx = idx / span, j = idx - pidx * span;
      wp_s[idx] = A.wparam[pidx * A.M + w_first + j];
    }
    __syncthreads();
    if (active) pl.load(P, wp_s, span, w - w_first, true);
    __syncthreads();                                         // wp_s is reused for the record tiles below
  } else if (active) {
    pl.load(P, A.wparam, A.M, w, (OPT & OPT_RANDP) != 0);
  }

  // record-slot table: slot r of this call holds the state after step (s0 / record_every + 1 + r) * record_every
  if (i == 0 && A.record_every > 0) {
    const uint32_t first_mult = s0 / (uint32_t)A.record_every + 1u;
    for (int r = 0; r < A.n_rec_cap && rec0 + (uint32_t)r < (uint32_t)kRecTableCap; ++r)
      A.rec_table[rec0 + r] = (first_mult + (uint32_t)r) * (uint32_t)A.record_every;
  }

  if (active) {
    float x[D];
    float iR[3] = { 0, 0, 0 }, ip[3] = { 0, 0, 0 }, att_cmd[4] = { 0, 0, 0, 0 }, rpm_cmd[4] = { 0, 0, 0, 0 };
    float target[4] = { 0, 0, 0, 0 };
    float md2[kMaxObst];
    const bool obst = (OPT & OPT_OBST) != 0 && (!GEN || A.min_d2 != nullptr);
    const bool ar = (OPT & OPT_AR) != 0 && (!GEN || A.eps != nullptr);                 // temporally correlated noise (R25)
    const bool costing = (OPT & OPT_COST) != 0 && (!GEN || A.cost_run != nullptr);     // R27
    const bool noise = (OPT & OPT_NOISE) != 0 && (!GEN || P.use_noise);                // compiled in AND requested
    const bool dist = (OPT & OPT_DIST) != 0 && (!GEN || P.dist_sigma > 0.0f);
    float eps[4] = { 0, 0, 0, 0 };
    float cost = 0.0f;
    if (A.bcast != nullptr) {
      // lazy cf_set_state(broadcast): every drone starts from the same state (uniform loads), controller integrals 0,
      // held commands = hover, obstacle minima re-armed -- nothing is read from the planes
#pragma unroll
      for (int j = 0; j < D; ++j) x[j] = A.bcast[j];
      att_cmd[3] = P.hover_thrust;
#pragma unroll
      for (int j = 0; j < 4; ++j) rpm_cmd[j] = P.hover_rpm;
#pragma unroll
      for (int j = 0; j < kMaxObst; ++j) md2[j] = __int_as_float(0x7f800000);
      eps[0] = __int_as_float(0x7fc00000);                     // NaN: the next command starts a fresh noise chain
    } else {
#pragma unroll
      for (int j = 0; j < D; ++j) x[j] = A.state[j * MN + i];
      if (ar) {
#pragma unroll
        for (int j = 0; j < 4; ++j) eps[j] = A.eps[j * MN + i];
      }
      if (costing) cost = A.cost_run[i];
      if (HAS_ATT) {
#pragma unroll
        for (int j = 0; j < 3; ++j) iR[j] = A.ctrl[j * MN + i];
      }
      if (HAS_POS) {
#pragma unroll
        for (int j = 0; j < 3; ++j) ip[j] = A.ctrl[(3 + j) * MN + i];
      }
      if (HAS_ATT || HAS_POS || !FP) {
#pragma unroll
        for (int j = 0; j < 4; ++j) att_cmd[j] = A.ctrl[(6 + j) * MN + i];
      }
      if (FP) {
#pragma unroll
        for (int j = 0; j < 4; ++j) rpm_cmd[j] = A.ctrl[(10 + j) * MN + i];
      }
      if (obst) {
#pragma unroll
        for (int j = 0; j < kMaxObst; ++j)      // registers hold min_t(|p|^2 - 2 c.p); |c|^2 is added back at the end
        md2[j] = j < P.n_obst ? A.min_d2[j * MN + i] - P.obst_q[j].w : __int_as_float(0x7f800000);
      }
    }
    float Rd[3][3];
    if (HAS_ATT) euler_to_R(att_cmd[0], att_cmd[1], att_cmd[2], Rd);
    // abstracted model, lean Euler step: the held attitude command folded with the step length (integrate_ab_euler_lean)
    constexpr bool AB_LEAN = !FP && INTEG == INTEG_EULER && !(OPT & OPT_EXTRAS);
    float held[4] = { 0, 0, 0, 0 };
    auto fold_command = [&]() {
      if constexpr (AB_LEAN) {
#pragma unroll
        for (int j = 0; j < 3; ++j) held[j] = pl.hc[j] * att_cmd[j];
        held[3] = pl.hct * att_cmd[3];
      }
    };
    fold_command();

    const uint32_t wg = (uint32_t)(w + A.world_offset), nn = (uint32_t)n;
    uint32_t s = s0;
    int att_phase = (int)(s0 % (uint32_t)P.att_div), pos_phase = (int)(s0 % (uint32_t)P.pos_div);
    int rec_phase = A.record_every > 0 ? (int)(s0 % (uint32_t)A.record_every) : 0;
    int rec_slot = 0;
    const int lane = threadIdx.x & 31;
    // record staging (REC_TMA): the warp's snapshots go to a [rec_group * D][32] tile (kRecBufs of them, used in turn); one
    // cp.async.bulk.tensor.2d of the whole tile by lane 0, box = 32 columns x rec_group * D rows at (column = first drone
    // of the warp, row = first slot of the group * D) of the [n_rec * D][MN] record tensor
    const int rec_group = REC == REC_PAIR ? 2 : A.rec_group;
    float *rec_tile = wp_s + warp_u * (kRecBufs * rec_group * D * 32);
    const uint32_t rec_tile_sa = (uint32_t)__cvta_generic_to_shared(wp_s) + (uint32_t)warp_u * (kRecBufs * rec_group * D * 128);
    const int rec_col = (int)blk0 + warp_u * 32;
    int rec_buf = 0, rec_grp = 0;
    // commands.  Buffer mode: one float4 per drone and command, prefetched one command ahead.  Noise mode: the nominal
    // sequence of this world's controller (R26), the same 16 bytes for (nearly) every lane: a plain indexed read-only
    // load at the top of the step, served by L1, with the Philox rounds between it and its use.
    const float4 *cp = noise ? A.cmds + (A.worlds_per_ctrl > 0 ? (w / A.worlds_per_ctrl) * A.n_cmds : 0)
                             : A.cmds + i;
    int cmds_left = (A.n_steps + A.cmd_hold - 1) / A.cmd_hold;  // commands this call consumes
    int cmd_k = 0;
    float4 next_cmd = make_float4(0.f, 0.f, 0.f, 0.f);
    if (!noise) next_cmd = __ldg(cp);
    // Software-pipelined random draws.  A Philox block + Box-Muller is a ~60-instruction serial chain that depends on
    // nothing but the counter, so the draw for the NEXT step is issued in the same basic block as this step's
    // integration: two independent chains for the scheduler to interleave (the kernel runs at 3-4 warps per
    // scheduler, where instruction-level parallelism inside a warp is what fills the issue slots).  zn holds the
    // normals of the next command (flat loop: a command every step), fdn the disturbance of the next step.
    const bool flat = A.cmd_hold == 1;
    float zn[4] = { 0, 0, 0, 0 }, fdn[3] = { 0, 0, 0 };
    auto draw4 = [&](uint32_t step, int stream, float *z) {
      uint32_t r[4];
      philox4x32_10_rk(A.rk, wg, nn, step, stream, r);
      normal_pair(r[0], r[1], z[0], z[1]);
      normal_pair(r[2], r[3], z[2], z[3]);
    };
    if (noise && flat) draw4(s0, STREAM_NOISE, zn);
    if (dist) {
      float z[4];
      draw4(s0, STREAM_DIST, z);
#pragma unroll
      for (int j = 0; j < 3; ++j) fdn[j] = P.dist_sigma * z[j];
    }

    // (1) command fetch
    auto fetch_command = [&](auto piped_c) {
      {
        float c[4];
        if (noise) {
          const float4 c4 = __ldg(cp + cmd_k);
          ++cmd_k;
          c[0] = c4.x; c[1] = c4.y; c[2] = c4.z; c[3] = c4.w;
          float z[4];
          if constexpr (decltype(piped_c)::value) {          // flat loop: drawn one step ahead; draw the next one now
#pragma unroll
            for (int j = 0; j < 4; ++j) z[j] = zn[j];
            draw4(s + 1u, STREAM_NOISE, zn);
          } else {
            draw4(s, STREAM_NOISE, z);
          }
          if (ar) {                                            // eps <- z (fresh chain) or beta eps + sqrt(1-beta^2) z
            const bool fresh = eps[0] != eps[0];
#pragma unroll
            for (int j = 0; j < 4; ++j) { eps[j] = fresh ? z[j] : fmaf(P.noise_beta, eps[j], P.noise_gain * z[j]); z[j] = eps[j]; }
          }
#pragma unroll
          for (int j = 0; j < 4; ++j) c[j] = clipf(fmaf(P.noise_sigma[j], z[j], c[j]), P.cmd_lo[j], P.cmd_hi[j]);
        } else {
          const float4 c4 = next_cmd;
          if constexpr (decltype(piped_c)::value) {
            // flat loop (a command every step): no branch -- the pointer stays on the last command (a harmless re-load)
            // and the L2 prefetch on a line that has been read
            --cmds_left;
            cp += cmds_left > 0 ? MN : 0;
            next_cmd = __ldg(cp);
            asm volatile("prefetch.global.L2 [%0];" :: "l"(cp + (cmds_left > 4 ? 4 * MN : 0)));
          } else
          if (--cmds_left > 0) {
            cp += MN;
            next_cmd = __ldg(cp);
            // a fresh command every step streams 16 bytes per drone and step from HBM (configs[2] variant 3B): one
            // step of cover does not hide DRAM latency at 16 warps per SM, so the line four commands ahead is pulled
            // into L2 now and the register prefetch above hits there
            if (flat && cmds_left > 4) asm volatile("prefetch.global.L2 [%0];" :: "l"(cp + 4 * MN));
          }
          c[0] = c4.x; c[1] = c4.y; c[2] = c4.z; c[3] = c4.w;
        }
        if (IFACE == IF_ATTITUDE) {
#pragma unroll
          for (int j = 0; j < 4; ++j) att_cmd[j] = c[j];
          if (HAS_ATT) euler_to_R(att_cmd[0], att_cmd[1], att_cmd[2], Rd);
          fold_command();
        } else if (IFACE == IF_POSITION) {
#pragma unroll
          for (int j = 0; j < 4; ++j) target[j] = c[j];
        } else if (IFACE == IF_ROTOR) {
#pragma unroll
          for (int j = 0; j < 4; ++j) rpm_cmd[j] = clipf(c[j], P.rpm_min, P.rpm_max);
        } else {   // torque interface: (tau_x, tau_y, tau_z, F) straight into the mixer
          mixer<OPT>(P, c[3], c, rpm_cmd);
        }
      }
    };
    // (8) record the current state (the caller has decided that a record is due)
    auto record_now = [&]() {
      const int rec_mode = REC == REC_RUNTIME ? A.rec_mode : RECB;
      if (rec_slot < A.n_rec_cap) {
        if (rec_mode == REC_TMA) {
          // Consecutive record slots are consecutive row blocks of the record tensor, so K = A.rec_group snapshots
          // are parked in one [K * D][32] tile and leave with ONE bulk-tensor store: the fence, the elected-lane
          // issue and its scoreboard waits are paid once per K records.  Two such tiles alternate.
          if (rec_grp == 0) {
            tma_store_wait_read<kRecBufs - 1>();  // the engine has read the tile handed over two groups ago
            __syncwarp();
          }
          float *t = rec_tile + (rec_buf * A.rec_group + rec_grp) * (D * 32);
#pragma unroll
          for (int j = 0; j < D; ++j) t[j * 32 + lane] = x[j];
          if (++rec_grp == A.rec_group) {
            fence_proxy_async_smem();             // generic-proxy writes -> visible to the async proxy
            __syncwarp();
            // first slot and buffer index as provably warp-uniform values (one shuffle): the TMA instruction takes
            // its operands from uniform registers; without this the compiler wraps it in a per-lane uniformisation loop
            const int sb = __shfl_sync(0xffffffffu, kRecBufs * (rec_slot + 1 - rec_grp) + rec_buf, 0);
            tma_store_tile_2d(&A.rec_map, rec_tile_sa + (sb % kRecBufs) * (A.rec_group * D * 128), rec_col,
                              (sb / kRecBufs) * D, lane == 0);
            rec_buf = (rec_buf + 1) % kRecBufs;
            rec_grp = 0;
          }
        } else {                                  // one streaming 4-byte store per component (any MN, any alignment)
          float *r = A.record + (size_t)rec_slot * D * MN + i;
#pragma unroll
          for (int j = 0; j < D; ++j) __stcs(r + j * MN, x[j]);
        }
      }
      ++rec_slot;
    };
    // (2)-(8) of one physics step
    float sn_t[3] = { 0, 0, 0 }, cs_t[3] = { 1, 1, 1 };     // sin / cos taken by a hoisted position tick, reused by the step that follows
    // hoist_c: the caller runs the position tick and the record test outside the step (position-interface loop below)
    auto physics_step = [&](auto obst_in_smem, auto fetch_c, auto pair_c, auto trig_c, auto hoist_c) {
      constexpr int PH = decltype(pair_c)::value;        // REC_PAIR: 0 / 1 = first / second step of a pair; else -1
      const int rec_mode = REC == REC_RUNTIME ? A.rec_mode : RECB;
      // sin / cos of the pre-step Euler angles (abstracted model, lean Euler step): taken first -- its range check is the
      // only data-dependent branch of the step -- and shared by the position tick and the integration
      float sn[3], cs[3];
      if constexpr (AB_LEAN) {
        if constexpr (decltype(trig_c)::value == 2) {                           // the position tick just took them (same state)
#pragma unroll
          for (int j = 0; j < 3; ++j) { sn[j] = sn_t[j]; cs[j] = cs_t[j]; }
        } else if constexpr (decltype(trig_c)::value == 1) {                    // the caller has bounded the run's angles
#pragma unroll
          for (int j = 0; j < 3; ++j) { sn[j] = mufu_sin(x[3 + j]); cs[j] = mufu_cos(x[3 + j]); }
        } else if constexpr (decltype(fetch_c)::value) sincos3_any(x + 3, sn, cs);     // flat loop: branch-free
        else sincos3_step(x + 3, sn, cs);
      }
      // (1) flat loop: this step's command (formed after the sin / cos so that everything below is one basic block)
      if constexpr (decltype(fetch_c)::value) fetch_command(IntC<1>{});
      // (2) position controller tick
      if (HAS_POS && !decltype(hoist_c)::value) {
        if (pos_phase == 0) {
          float zB[3];
          if (FP) {
            const float *q = x + 3;
            zB[0] = 2.0f * (q[0] * q[2] + q[3] * q[1]);
            zB[1] = 2.0f * (q[1] * q[2] - q[3] * q[0]);
            zB[2] = 1.0f - 2.0f * (q[0] * q[0] + q[1] * q[1]);
          } else {
            if constexpr (!AB_LEAN) sincos3_step(x + 3, sn, cs);
            zB[0] = cs[2] * sn[1] * cs[0] + sn[2] * sn[0]; zB[1] = sn[2] * sn[1] * cs[0] - cs[2] * sn[0];
            zB[2] = cs[1] * cs[0];
          }
          position_tick(P, x, FP ? x + 7 : x + 6, zB, target, ip, att_cmd);
          if (HAS_ATT) euler_to_R(att_cmd[0], att_cmd[1], att_cmd[2], Rd);
          fold_command();
        }
        pos_phase = pos_phase + 1 == P.pos_div ? 0 : pos_phase + 1;
      }
      // (3) attitude controller tick + mixer
      if (HAS_ATT) {
        if constexpr (PH == 0) {
          attitude_tick<OPT>(P, x + 3, x + 10, Rd, att_cmd[3], iR, rpm_cmd);
        } else if constexpr (PH < 0) {
          if (att_phase == 0) attitude_tick<OPT>(P, x + 3, x + 10, Rd, att_cmd[3], iR, rpm_cmd);
          att_phase = att_phase + 1 == P.att_div ? 0 : att_phase + 1;
        }
      }
      // (4) disturbance of this step (drawn one step ahead, held over the RK4 stages) and the draw for the next step
      float fdist[3] = { 0, 0, 0 };
      if (dist) {
        float z[4];
#pragma unroll
        for (int j = 0; j < 3; ++j) fdist[j] = fdn[j];
        draw4(s + 1u, STREAM_DIST, z);
#pragma unroll
        for (int j = 0; j < 3; ++j) fdn[j] = P.dist_sigma * z[j];
      }
      // (5) integrate, (6) count
      integrate<MODEL, INTEG, OPT>(P, pl, x, FP ? rpm_cmd : att_cmd, fdist, held, sn, cs);
      ++s;
      // (7) obstacle minima (squared centre distance; the square roots are taken once, at read-out)
      if (obst) {
        // |p - c_j|^2 = (|p|^2 - 2 c_j.p) + |c_j|^2, and the constant |c_j|^2 commutes with the minimum over time: the
        // registers track min_t(|p|^2 - 2 c_j.p) with 3 FFMA + FMNMX per sphere and step, |c_j|^2 is added once when
        // the minima leave the registers (unused slots: + inf, they never win)
        float pp = fmaf(x[2], x[2], fmaf(x[1], x[1], x[0] * x[0]));
#pragma unroll
        for (int j = 0; j < kMaxObst; ++j) {
          float qx, qy, qz;
          if constexpr (decltype(obst_in_smem)::value) { const float4 oq = obst_s[j]; qx = oq.x; qy = oq.y; qz = oq.z; }
          else { qx = P.obst_x[j]; qy = P.obst_y[j]; qz = P.obst_z[j]; }
          md2[j] = fminf(md2[j], fmaf(qz, x[2], fmaf(qy, x[1], fmaf(qx, x[0], pp))));
        }
      }
      // (7b) running rollout cost on the post-step state (R27): h w_pos |p - goal|^2 + h w_vel |v|^2
      if (costing) {
        const float *v = FP ? x + 7 : x + 6;
        float ex = x[0] - P.cost_goal[0], ey = x[1] - P.cost_goal[1], ez = x[2] - P.cost_goal[2];
        float e2 = fmaf(ez, ez, fmaf(ey, ey, ex * ex)), v2 = fmaf(v[2], v[2], fmaf(v[1], v[1], v[0] * v[0]));
        cost = fmaf(P.cost_hw_pos, e2, fmaf(P.cost_hw_vel, v2, cost));
      }
      // (8) record
      if constexpr (PH >= 0 && REC == REC_PAIR) {   // REC_PAIR: every step recorded, two snapshots per store, no test
        if constexpr (PH == 0) {
          tma_store_wait_read<kRecBufs - 1>();      // the engine has read the tile handed over two pairs ago
          __syncwarp();
        }
        float *t = rec_tile + (rec_buf * 2 + PH) * (D * 32);
#pragma unroll
        for (int j = 0; j < D; ++j) t[j * 32 + lane] = x[j];
        if constexpr (PH == 1) {
          fence_proxy_async_smem();
          __syncwarp();
          const int sb = __shfl_sync(0xffffffffu, kRecBufs * rec_slot + rec_buf, 0);
          tma_store_tile_2d(&A.rec_map, rec_tile_sa + (sb % kRecBufs) * (2 * D * 128), rec_col, (sb / kRecBufs) * D, lane == 0);
          rec_buf ^= 1;
          rec_slot += 2;
        }
      } else
      if constexpr (!decltype(hoist_c)::value) {
        if (rec_mode != REC_NONE) {
          if (++rec_phase == A.record_every) {
            rec_phase = 0;
            record_now();
          }
        }
      }
    };
    // unroll factors measured on the branch-free loop bodies (1 / 2 / 4 / 5): the per-step-command loop x2 with in-kernel
    // noise commands, x4 with a command buffer (cfg3b +2 %); the bounded held-command loop x2 (planner rollout +2.3 %)
    constexpr int kUnrollFlat = (OPT & OPT_NOISE) ? 2 : 4;
    // The call starts at a command boundary (C8), so a run of cmd_hold steps starts with ONE command fetch.  With held
    // commands the loop is two-level and the inner loop carries no command logic (mppi rollout kernel 705 -> 691 us,
    // cfg4 +3 %); with a fresh command every step (cmd_hold == 1, configs[2]) the flat loop is 2 % faster.
    if (flat) {
#pragma unroll kUnrollFlat
      for (int t = 0; t < A.n_steps; ++t) physics_step(NoSmem{}, IntC<1>{}, IntC<-1>{}, IntC<0>{}, IntC<0>{});
    } else if constexpr (PAIRED) {
      const bool rec_each = RECB != REC_NONE && A.record_every == 1;
      for (int t = 0; t < A.n_steps;) {
        fetch_command(IntC<0>{});
        const int run_len = A.n_steps - t < A.cmd_hold ? A.n_steps - t : A.cmd_hold;     // even (host)
        t += run_len;
        for (int k = 0; k < run_len; k += 2) {
          if constexpr (REC == REC_PAIR) {
            physics_step(InSmem{}, IntC<0>{}, IntC<0>{}, IntC<0>{}, IntC<0>{});
            physics_step(InSmem{}, IntC<0>{}, IntC<1>{}, IntC<0>{}, IntC<0>{});
          } else {                                  // record test between the steps (every step) / after the pair (even period)
            physics_step(InSmem{}, IntC<0>{}, IntC<0>{}, IntC<0>{}, IntC<1>{});
            if (RECB != REC_NONE && rec_each) record_now();
            physics_step(InSmem{}, IntC<0>{}, IntC<1>{}, IntC<0>{}, IntC<1>{});
            if (RECB != REC_NONE) {
              rec_phase += 2;
              if (rec_each || rec_phase == A.record_every) { rec_phase = 0; record_now(); }
            }
          }
        }
      }
    } else {
      for (int t = 0; t < A.n_steps;) {
        fetch_command(IntC<0>{});
        const int run_len = A.n_steps - t < A.cmd_hold ? A.n_steps - t : A.cmd_hold;
        t += run_len;
        if constexpr (AB_LEAN && IFACE == IF_ATTITUDE) {
          // Held command (abstracted model, attitude interface): the sin / cos range test is taken for the whole run
          // from a bound on how far the angles can move while this command is held: with P = max_j |Psi_j|,
          // Q = max_j |dPsi_j|, C = max_j |h c_j u_j| the Euler step of Eq. (10) gives P+ <= P + h Q,
          // Q+ <= max|1 + h b| Q + max|h a| P + C (2 FFMA per step of the run).  Within 6.28 (the margin covers the
          // rounding of the recursion) the run takes the test-free loop body.
          bool bounded = A.ang_bound_ok != 0 && run_len <= 32;
          if (bounded) {
            float Pm = fmaxf(fmaxf(fabsf(x[3]), fabsf(x[4])), fabsf(x[5])), Qm = fmaxf(fmaxf(fabsf(x[9]), fabsf(x[10])), fabsf(x[11]));
            const float C = fmaxf(fmaxf(fabsf(held[0]), fabsf(held[1])), fabsf(held[2]));
            for (int k = 0; k < run_len; ++k) {
              const float Pn = fmaf(P.h, Qm, Pm);
              Qm = fmaf(P.bnd_hb1, Qm, fmaf(P.bnd_ha, Pm, C));
              Pm = Pn;
            }
            bounded = Pm <= 6.28f;                  // NaN -> false
          }
          if (bounded) {
#pragma unroll 2
            for (int k = 0; k < run_len; ++k) physics_step(InSmem{}, IntC<0>{}, IntC<-1>{}, IntC<1>{}, IntC<0>{});
          } else {
            for (int k = 0; k < run_len; ++k) physics_step(InSmem{}, IntC<0>{}, IntC<-1>{}, IntC<0>{}, IntC<0>{});
          }
        } else if constexpr (AB_LEAN && IFACE == IF_POSITION) {
          // Position interface (configs[3]): the run is cut into sub-runs that end at the next position tick or the next
          // record, whichever comes first, so that the tick (which sets the attitude command the sub-run holds), the
          // record test and the angle bound sit BETWEEN sub-runs and the inner loop body has no branch left.
          const int rec_mode = REC == REC_RUNTIME ? A.rec_mode : RECB;
          for (int k = 0; k < run_len;) {
            const bool ticked = pos_phase == 0;
            if (ticked) {                                             // (2) position tick on this step's pre-step state
              float zB[3];
              sincos3_step(x + 3, sn_t, cs_t);
              zB[0] = cs_t[2] * sn_t[1] * cs_t[0] + sn_t[2] * sn_t[0]; zB[1] = sn_t[2] * sn_t[1] * cs_t[0] - cs_t[2] * sn_t[0];
              zB[2] = cs_t[1] * cs_t[0];
              position_tick(P, x, x + 6, zB, target, ip, att_cmd);
              fold_command();
            }
            int sub = run_len - k;
            if (P.pos_div - pos_phase < sub) sub = P.pos_div - pos_phase;
            if (rec_mode != REC_NONE && A.record_every - rec_phase < sub) sub = A.record_every - rec_phase;
            bool bounded = A.ang_bound_ok != 0 && sub <= 32;
            if (bounded) {
              float Pm = fmaxf(fmaxf(fabsf(x[3]), fabsf(x[4])), fabsf(x[5])), Qm = fmaxf(fmaxf(fabsf(x[9]), fabsf(x[10])), fabsf(x[11]));
              const float C = fmaxf(fmaxf(fabsf(held[0]), fabsf(held[1])), fabsf(held[2]));
              for (int j = 0; j < sub; ++j) {
                const float Pn = fmaf(P.h, Qm, Pm);
                Qm = fmaf(P.bnd_hb1, Qm, fmaf(P.bnd_ha, Pm, C));
                Pm = Pn;
              }
              bounded = Pm <= 6.28f;
            }
            int j0 = 0;
            if (ticked) { physics_step(InSmem{}, IntC<0>{}, IntC<-1>{}, IntC<2>{}, IntC<1>{}); j0 = 1; }   // the tick's sin / cos
            if (bounded) {
              for (int j = j0; j < sub; ++j) physics_step(InSmem{}, IntC<0>{}, IntC<-1>{}, IntC<1>{}, IntC<1>{});
            } else {
              for (int j = j0; j < sub; ++j) physics_step(InSmem{}, IntC<0>{}, IntC<-1>{}, IntC<0>{}, IntC<1>{});
            }
            k += sub;
            pos_phase += sub;
            if (pos_phase == P.pos_div) pos_phase = 0;
            if (rec_mode != REC_NONE) {
              rec_phase += sub;
              if (rec_phase == A.record_every) { rec_phase = 0; record_now(); }
            }
          }
        } else {
          for (int k = 0; k < run_len; ++k) physics_step(InSmem{}, IntC<0>{}, IntC<-1>{}, IntC<0>{}, IntC<0>{});
        }
      }
    }
    if (RECB == REC_TMA || REC == REC_PAIR || (REC == REC_RUNTIME && A.rec_mode == REC_TMA)) {
      if (REC != REC_PAIR && rec_grp > 0) {                              // a partial last group leaves record by record (box = D rows)
        fence_proxy_async_smem();
        __syncwarp();
        const int sb = __shfl_sync(0xffffffffu, kRecBufs * (rec_slot - rec_grp) + rec_buf, 0);
        const int n_tail = __shfl_sync(0xffffffffu, rec_grp, 0);
        for (int r = 0; r < n_tail; ++r)
          tma_store_tile_2d(&A.rec_map1, rec_tile_sa + ((sb % kRecBufs) * A.rec_group + r) * (D * 128), rec_col,
                            (sb / kRecBufs + r) * D, lane == 0);
      }
      tma_store_wait_read<0>();                       // the tiles must outlive the engine's reads
      __syncwarp();
    }
    // final store
#pragma unroll
    for (int j = 0; j < D; ++j) A.state[j * MN + i] = x[j];
    if (HAS_ATT) {
#pragma unroll
      for (int j = 0; j < 3; ++j) A.ctrl[j * MN + i] = iR[j];
    }
    if (HAS_POS) {
#pragma unroll
      for (int j = 0; j < 3; ++j) A.ctrl[(3 + j) * MN + i] = ip[j];
    }
    if (HAS_ATT || HAS_POS || !FP) {
#pragma unroll
      for (int j = 0; j < 4; ++j) A.ctrl[(6 + j) * MN + i] = att_cmd[j];
    }
    if (FP) {
#pragma unroll
      for (int j = 0; j < 4; ++j) A.ctrl[(10 + j) * MN + i] = rpm_cmd[j];
    }
    float d_min = __int_as_float(0x7f800000);
    if (obst) {
#pragma unroll
      for (int j = 0; j < kMaxObst; ++j) { md2[j] += P.obst_q[j].w; A.min_d2[j * MN + i] = md2[j]; }
      if (A.md_drone != nullptr || costing) {   // C10 read-out fused into the epilogue: min_j sqrt(min_t d2_j) - r_j
#pragma unroll
        for (int j = 0; j < kMaxObst; ++j)
          if (j < P.n_obst) d_min = fminf(d_min, sqrtf(md2[j]) - P.obst[j][3]);
        if (A.md_drone != nullptr) A.md_drone[i] = d_min;
      }
    }
    if (ar) {
#pragma unroll
      for (int j = 0; j < 4; ++j) A.eps[j * MN + i] = eps[j];
    }
    if (costing) {       // R27 read-out: J = J_run + w_term |p - goal|^2 + w_obs max(0, d_safe - d_min)^2 + w_coll [d_min < 0]
      A.cost_run[i] = cost;
      float ex = x[0] - P.cost_goal[0], ey = x[1] - P.cost_goal[1], ez = x[2] - P.cost_goal[2];
      float J = fmaf(P.cost_w_term, fmaf(ez, ez, fmaf(ey, ey, ex * ex)), cost);
      float gap = P.cost_d_safe - d_min;
      if (gap > 0.0f) J = fmaf(P.cost_w_obs * gap, gap, J);
      if (d_min < 0.0f) J += P.cost_w_coll;
      A.cost_drone[i] = J;
    }
  }
  // the last block to finish advances the device-side counters (every block has read s0 by then), so that a captured
  // CUDA graph of single-step launches replays correctly.  Controller ticks happen at the steps s in [s0, s0 + n) with
  // s % div == 0: a closed form, nothing is counted in the loop.
  if (threadIdx.x == 0) {
    __threadfence();
    uint32_t done = atomicAdd(&A.counters->blocks_done, 1u);
    if (SLICED && done == gridDim.x - 1 && !A.advance) A.counters->blocks_done = 0;   // a slice that is not the call's last one
    if (done == gridDim.x - 1 && (!SLICED || A.advance)) {
      const uint32_t s1 = s0 + (uint32_t)A.n_steps;
      uint32_t n_rec = A.record_every > 0 ? s1 / (uint32_t)A.record_every - s0 / (uint32_t)A.record_every : 0u;
      auto ticks = [&](uint32_t div) { return (s1 + div - 1u) / div - (s0 + div - 1u) / div; };
      if (HAS_ATT) A.counters->att_ticks += ticks((uint32_t)P.att_div);
      if (HAS_POS) A.counters->pos_ticks += ticks((uint32_t)P.pos_div);
      A.counters->s = s1;
      A.counters->n_rec_total = rec0 + n_rec;
      A.counters->blocks_done = 0;
      __threadfence();
    }
  }
}

// launch table entry points, one translation unit per model (cf_rollout_fp.cu / cf_rollout_ab.cu)
struct LaunchCfg { int grid, block; size_t smem; cudaStream_t stream; };
// returns false if (integ, iface, opt) has no instantiation that covers it; *name = instantiation label, *opt_used
bool launch_fp(int integ, int iface, int opt, int rec_mode, const StepArgs *A, const DevParams *P, const LaunchCfg *L,
               const char **name, int *opt_used, bool dry);
bool launch_ab(int integ, int iface, int opt, int rec_mode, const StepArgs *A, const DevParams *P, const LaunchCfg *L,
               const char **name, int *opt_used, bool dry);

// shared by the two launch tables: the entry that serves (integ, iface, opt, rec_mode), or nullptr
struct RolloutEntry { int integ, iface, opt, rec; const char *name; void (*fn)(const StepArgs, const DevParams); };
inline const RolloutEntry *pick_rollout(const RolloutEntry *tab, int n, int integ, int iface, int opt, int rec_mode) {
  const RolloutEntry *best = nullptr;
  for (int k = 0; k < n; ++k) {
    const RolloutEntry &e = tab[k];
    if (e.integ != integ || e.iface != iface || (e.opt & opt) != opt) continue;
    // a lean kernel takes its options as unconditionally on: it serves only requests with exactly its options
    // (OPT_RANDP may be extra: the parameter planes always hold valid values) and exactly its record mode
    if (!(e.opt & OPT_EXTRAS) && ((e.opt & ~OPT_RANDP) != (opt & ~OPT_RANDP) || e.rec != rec_mode)) continue;
    if (!best || __builtin_popcount(e.opt) < __builtin_popcount(best->opt)) best = &e;
  }
  return best;
}

}  // namespace cf
