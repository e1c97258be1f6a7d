// cf_grad.cu -- reverse-mode differentiation of the fused rollout (Fig. 3D: "differentiating a goal
// distance with respect to the control inputs" through n consecutive steps, dynamics AND onboard controller stack).
//
//   L(u) = || p_n(u) - goal ||,   g[k] = dL / du[k]   for the command sequence u[k] (each held cmd_hold steps),
//
// as one hand-written adjoint kernel in two launches (no tape, no autodiff framework): thread = drone.  Forward sweep: the production
// step (same device functions as the rollout kernel: deriv_fp / deriv_ab, attitude_tick, mixer) with the pre-step state
// of every step parked in a caller-provided history buffer [n_steps][HD][MN] (SoA, coalesced).  Backward sweep: for
// t = n-1 .. 0 the step is recomputed from its parked state and the cotangent is pulled back through quaternion
// normalisation, RK4 / Euler (stage states recomputed in registers), the derivative (hand-derived VJPs of Eqs. (1)-(4),
// (6) and (7)-(10)), the motor mixer (sqrt and clips: derivative 0 where a clip is active, reading R33) and the attitude
// controller (rotation-matrix error, clipped integral, desired rotation from the commanded Euler angles).  The adjoint
// of a held command accumulates over the steps / ticks that used it and is written when its fetch step is reached.
// The simulator state is not modified.  Configurations with fidelity extras, force disturbances or the torque interface run
// the GENERAL instantiations (OPT = GOPT): generic integrator and 17 / 13-wide pull-back, VJPs of full Eq. (6), the thrust
// / torque polynomials, Eq. (5), body drag and the simplified abstracted model, the disturbance re-drawn from Philox.
#include "cf_internal.h"

using namespace cf;

namespace {

struct GradArgs {
  const float *state, *ctrl, *wparam;
  const float4 *cmds;      // [n_cmds][MN]
  float4 *grad;            // [n_cmds][MN]
  float *loss;             // [MN]
  float4 *hist;            // [n_steps][HD / 4][MN] float4
  long long MN, M, N;
  int n_steps, cmd_hold, n_cmds;
  uint32_t s0;
  float goal[3];
  long long world_offset;
  uint32_t rk[20];         // Philox round keys of the simulator's seed (general kernels: the DIST stream)
};

template <int MODEL> struct Dim { static constexpr int D = MODEL == MODEL_FP ? 17 : 13; };

// ---- VJP of the first-principles derivative (lean form: Eq. (6) with one time constant, pure-quadratic curves) -------
// cotangent a[17] of dx -> gx[17] (accumulated into), gu[4] (accumulated into)
__device__ __forceinline__ void vjp_deriv_fp(const DevParams &P, const Plant<MODEL_FP, 0> &pl, const float *x,
                                             const float *a, float *gx, float *gu) {
  const float *q = x + 3, *w = x + 10, *Om = x + 13;
  const float *a_p = a, *a_q = a + 3, *a_v = a + 7, *a_w = a + 10, *a_Om = a + 13;
  float *g_q = gx + 3, *g_v = gx + 7, *g_w = gx + 10, *g_Om = gx + 13;
#pragma unroll
  for (int j = 0; j < 3; ++j) g_v[j] += a_p[j];                                       // Eq. (1)
  // Eq. (3): dv = zB F/m - g e_z
  float w2s = Om[0] * Om[0] + Om[1] * Om[1] + Om[2] * Om[2] + Om[3] * Om[3];
  float acc = pl.kf2 * w2s * pl.inv_m;
  float zx = 2.0f * (q[0] * q[2] + q[3] * q[1]), zy = 2.0f * (q[1] * q[2] - q[3] * q[0]);
  float zz = 1.0f - 2.0f * (q[0] * q[0] + q[1] * q[1]);
  float gF = (zx * a_v[0] + zy * a_v[1] + zz * a_v[2]) * pl.inv_m;
  float gzx = a_v[0] * acc, gzy = a_v[1] * acc, gzz = a_v[2] * acc;
  g_q[0] += 2.0f * (q[2] * gzx - q[3] * gzy) - 4.0f * q[0] * gzz;
  g_q[1] += 2.0f * (q[3] * gzx + q[2] * gzy) - 4.0f * q[1] * gzz;
  g_q[2] += 2.0f * (q[0] * gzx + q[1] * gzy);
  g_q[3] += 2.0f * (q[1] * gzx - q[0] * gzy);
  // Eq. (4): dw = tau/J + cJ (w x w terms); tau from the mixing matrix C1
  float gt[3] = { a_w[0] * pl.inv_J[0], a_w[1] * pl.inv_J[1], a_w[2] * pl.inv_J[2] };
  const float lk = P.lever * pl.kf2;
  const float sx[4] = { -1, -1, 1, 1 }, sy[4] = { -1, 1, 1, -1 }, sz[4] = { -1, 1, -1, 1 };
#pragma unroll
  for (int k = 0; k < 4; ++k) {
    float g_w2 = pl.kf2 * gF + lk * (sx[k] * gt[0] + sy[k] * gt[1]) + pl.km2 * sz[k] * gt[2];
    g_Om[k] += 2.0f * Om[k] * g_w2 - pl.cv * a_Om[k];                                 // Eq. (6): dOm = cv (u - Om)
    gu[k] += pl.cv * a_Om[k];
  }
  g_w[1] += pl.cJ[0] * w[2] * a_w[0]; g_w[2] += pl.cJ[0] * w[1] * a_w[0];
  g_w[2] += pl.cJ[1] * w[0] * a_w[1]; g_w[0] += pl.cJ[1] * w[2] * a_w[1];
  g_w[0] += pl.cJ[2] * w[1] * a_w[2]; g_w[1] += pl.cJ[2] * w[0] * a_w[2];
  // Eq. (2): dq = 1/2 q (x) (w, 0)
  float bx = 0.5f * a_q[0], by = 0.5f * a_q[1], bz = 0.5f * a_q[2], bw = 0.5f * a_q[3];
  g_q[3] += w[0] * bx + w[1] * by + w[2] * bz;
  g_q[0] += -w[2] * by + w[1] * bz - w[0] * bw;
  g_q[1] += w[2] * bx - w[0] * bz - w[1] * bw;
  g_q[2] += -w[1] * bx + w[0] * by - w[2] * bw;
  g_w[0] += q[3] * bx + q[2] * by - q[1] * bz - q[0] * bw;
  g_w[1] += -q[2] * bx + q[3] * by + q[0] * bz - q[1] * bw;
  g_w[2] += q[1] * bx - q[0] * by + q[3] * bz - q[2] * bw;
}

// ---- VJP of the abstracted derivative, Eqs. (7)-(10) -------------------------------------------------------------------
__device__ __forceinline__ void vjp_deriv_ab(const DevParams &P, const Plant<MODEL_AB, 0> &pl, const float *x,
                                             const float *a, float *gx, float *gu) {
  float sn[3], cs[3];
  sincos3_step(x + 3, sn, cs);
  const float sr = sn[0], cr = cs[0], sp = sn[1], cp = cs[1], sy = sn[2], cy = cs[2];
  const float *a_p = a, *a_ps = a + 3, *a_v = a + 6, *a_dps = a + 9;
  const float a_f = a[12];
  float zx = cy * sp * cr + sy * sr, zy = sy * sp * cr - cy * sr, zz = cp * cr;
  float acc = (P.ab_cf * x[12]) * pl.inv_m;
#pragma unroll
  for (int j = 0; j < 3; ++j) {
    gx[6 + j] += a_p[j];                                                              // dp = v
    gx[9 + j] += a_ps[j] + pl.b[j] * a_dps[j];                                        // dPsi = dPsi ; Eq. (10)
    gx[3 + j] += pl.a[j] * a_dps[j];
    gu[j] += pl.c[j] * a_dps[j];
  }
  // dv = zB cf f/m - g e_z : angles through zB, thrust state through acc
  float dzr[3] = { -cy * sp * sr + sy * cr, -sy * sp * sr - cy * cr, -cp * sr };
  float dzp[3] = { cy * cp * cr, sy * cp * cr, -sp * cr };
  float dzy[3] = { -sy * sp * cr + cy * sr, cy * sp * cr + sy * sr, 0.0f };
  gx[3] += (dzr[0] * a_v[0] + dzr[1] * a_v[1] + dzr[2] * a_v[2]) * acc;
  gx[4] += (dzp[0] * a_v[0] + dzp[1] * a_v[1] + dzp[2] * a_v[2]) * acc;
  gx[5] += (dzy[0] * a_v[0] + dzy[1] * a_v[1]) * acc;
  gx[12] += (zx * a_v[0] + zy * a_v[1] + zz * a_v[2]) * (P.ab_cf * pl.inv_m) - pl.ctau * a_f;   // Eq. (9)
  gu[3] += pl.ctau * a_f;
}

// ---- shared pieces of the controller VJPs -----------------------------------------------------------------------------
// R = quat_to_R(q): cotangent GR[i][j] = dL/dR_ij -> g_q (accumulated)
__device__ __forceinline__ void vjp_quat_to_R(const float *q, const float GR[3][3], float *g_q) {
  const float x = q[0], y = q[1], z = q[2], ww = q[3];
  g_q[0] += 2.0f * (y * (GR[0][1] + GR[1][0]) + z * (GR[0][2] + GR[2][0]) + ww * (GR[2][1] - GR[1][2])) - 4.0f * x * (GR[1][1] + GR[2][2]);
  g_q[1] += 2.0f * (x * (GR[0][1] + GR[1][0]) + z * (GR[1][2] + GR[2][1]) + ww * (GR[0][2] - GR[2][0])) - 4.0f * y * (GR[0][0] + GR[2][2]);
  g_q[2] += 2.0f * (x * (GR[0][2] + GR[2][0]) + y * (GR[1][2] + GR[2][1]) + ww * (GR[1][0] - GR[0][1])) - 4.0f * z * (GR[0][0] + GR[1][1]);
  g_q[3] += 2.0f * (x * (GR[2][1] - GR[1][2]) + y * (GR[0][2] - GR[2][0]) + z * (GR[1][0] - GR[0][1]));
}
// Rd = Rz(yaw) Ry(pitch) Rx(roll) (reading R13) from its sines / cosines
__device__ __forceinline__ void euler_R_from_sc(const float *sn, const float *cs, float Rd[3][3]) {
  const float sr = sn[0], cr = cs[0], sp = sn[1], cp = cs[1], sy = sn[2], cy = cs[2];
  Rd[0][0] = cy * cp; Rd[0][1] = cy * sp * sr - sy * cr; Rd[0][2] = cy * sp * cr + sy * sr;
  Rd[1][0] = sy * cp; Rd[1][1] = sy * sp * sr + cy * cr; Rd[1][2] = sy * sp * cr - cy * sr;
  Rd[2][0] = -sp;     Rd[2][1] = cp * sr;                Rd[2][2] = cp * cr;
}
// cotangent GD[i][j] = dL/dRd_ij -> (roll, pitch, yaw) (accumulated): d/droll rotates columns 1, 2; d/dyaw rotates rows
// 0, 1; d/dpitch written out
__device__ __forceinline__ void vjp_euler_R(const float Rd[3][3], const float *sn, const float *cs, const float GD[3][3],
                                            float *g_ang) {
  const float sr = sn[0], cr = cs[0], sp = sn[1], cp = cs[1], sy = sn[2], cy = cs[2];
  g_ang[0] += GD[0][1] * Rd[0][2] - GD[0][2] * Rd[0][1] + GD[1][1] * Rd[1][2] - GD[1][2] * Rd[1][1] + GD[2][1] * Rd[2][2] - GD[2][2] * Rd[2][1];
  g_ang[1] += GD[0][0] * (-cy * sp) + GD[0][1] * (cy * cp * sr) + GD[0][2] * (cy * cp * cr)
            + GD[1][0] * (-sy * sp) + GD[1][1] * (sy * cp * sr) + GD[1][2] * (sy * cp * cr)
            + GD[2][0] * (-cp) + GD[2][1] * (-sp * sr) + GD[2][2] * (-sp * cr);
  g_ang[2] += -GD[0][0] * Rd[1][0] - GD[0][1] * Rd[1][1] - GD[0][2] * Rd[1][2]
            + GD[1][0] * Rd[0][0] + GD[1][1] * Rd[0][1] + GD[1][2] * Rd[0][2];
}
// ---- the general kernels (fidelity extras, disturbances, torque interface): option set of their device functions ------
constexpr int GOPT = OPT_EXTRAS | OPT_DIST;

// body drag  d = R (Ca . (R^T v)) / m  (Eq. (3) / Eq. (8) with C_a != 0): cotangent gd of d -> g_v (accumulated) and the
// cotangent GR of the rotation matrix (assigned)
__device__ __forceinline__ void vjp_drag(const DevParams &P, float inv_m, const float R[3][3], const float *v, const float *gd,
                                         float *g_v, float GR[3][3]) {
  float b[3], gc[3], gb[3];
#pragma unroll
  for (int j = 0; j < 3; ++j) {
    b[j] = R[0][j] * v[0] + R[1][j] * v[1] + R[2][j] * v[2];                         // body-frame velocity
    gc[j] = (R[0][j] * gd[0] + R[1][j] * gd[1] + R[2][j] * gd[2]) * inv_m;           // cotangent of c = Ca . b
    gb[j] = P.Ca[j] * gc[j];
  }
#pragma unroll
  for (int i = 0; i < 3; ++i) {
    g_v[i] += R[i][0] * gb[0] + R[i][1] * gb[1] + R[i][2] * gb[2];
#pragma unroll
    for (int j = 0; j < 3; ++j) GR[i][j] = gd[i] * inv_m * (P.Ca[j] * b[j]) + v[i] * gb[j];
  }
}

// ---- VJP of the first-principles derivative with the fidelity extras (deriv_fp<OPT_EXTRAS>): asymmetric + quadratic
// rotor dynamics (full Eq. (6)), thrust / torque polynomials, Eq. (5) gyroscopic and reaction torque (reading R2), body
// drag.  The disturbance force is additive and has no derivative.  u = held rotor command.
__device__ __forceinline__ void vjp_deriv_fp_ex(const DevParams &P, const Plant<MODEL_FP, GOPT> &pl, const float *x,
                                                const float *u, const float *a, float *gx, float *gu) {
  const float *q = x + 3, *v = x + 7, *w = x + 10, *Om = x + 13;
  const float *a_p = a, *a_q = a + 3, *a_v = a + 7, *a_w = a + 10, *a_Om = a + 13;
  float *g_q = gx + 3, *g_v = gx + 7, *g_w = gx + 10, *g_Om = gx + 13;
#pragma unroll
  for (int j = 0; j < 3; ++j) g_v[j] += a_p[j];                                       // Eq. (1)
  float f[4], dOm[4], cvk[4], cdk[4];
#pragma unroll
  for (int k = 0; k < 4; ++k) {
    float e = u[k] - Om[k];
    bool up = e >= 0.0f;
    cvk[k] = up ? pl.cv : pl.cv_dn; cdk[k] = up ? pl.cd_up : pl.cd_dn;
    dOm[k] = cvk[k] * e + cdk[k] * (u[k] * u[k] - Om[k] * Om[k]);
    f[k] = pl.kf0 + Om[k] * (pl.kf1 + pl.kf2 * Om[k]);
  }
  const float F = (f[0] + f[1]) + (f[2] + f[3]);
  // Eq. (3): dv = zB F/m + f_dist/m - g e_z (+ drag)
  float acc = F * pl.inv_m;
  float zx = 2.0f * (q[0] * q[2] + q[3] * q[1]), zy = 2.0f * (q[1] * q[2] - q[3] * q[0]);
  float zz = 1.0f - 2.0f * (q[0] * q[0] + q[1] * q[1]);
  float gF = (zx * a_v[0] + zy * a_v[1] + zz * a_v[2]) * pl.inv_m;
  float gzx = a_v[0] * acc, gzy = a_v[1] * acc, gzz = a_v[2] * acc;
  g_q[0] += 2.0f * (q[2] * gzx - q[3] * gzy) - 4.0f * q[0] * gzz;
  g_q[1] += 2.0f * (q[3] * gzx + q[2] * gzy) - 4.0f * q[1] * gzz;
  g_q[2] += 2.0f * (q[0] * gzx + q[1] * gzy);
  g_q[3] += 2.0f * (q[1] * gzx - q[0] * gzy);
  if (P.has_drag) {
    float R[3][3], GR[3][3];
    quat_to_R(q, R);
    vjp_drag(P, pl.inv_m, R, v, a_v, g_v, GR);
    vjp_quat_to_R(q, GR, g_q);
  }
  // Eq. (4): dw = tau/J + cJ (w x w terms); tau from the mixing matrix C1 (+ Eq. (5))
  float gt[3] = { a_w[0] * pl.inv_J[0], a_w[1] * pl.inv_J[1], a_w[2] * pl.inv_J[2] };
  float gS = 0.0f, gdS = 0.0f;
  if (P.has_gyro) {     // tau += Jp (-w_y S, +w_x S, -dS), S = W1 - W2 + W3 - W4 (rad/s)
    const float S = (Om[0] - Om[1]) + (Om[2] - Om[3]);
    g_w[1] -= P.Jp_rad * S * gt[0];
    g_w[0] += P.Jp_rad * S * gt[1];
    gS = P.Jp_rad * (w[0] * gt[1] - w[1] * gt[0]);
    gdS = -P.Jp_rad * gt[2];
  }
  const float sx[4] = { -1, -1, 1, 1 }, sy[4] = { -1, 1, 1, -1 }, sz[4] = { -1, 1, -1, 1 }, sd[4] = { 1, -1, 1, -1 };
#pragma unroll
  for (int k = 0; k < 4; ++k) {
    const float gfk = gF + P.lever * (sx[k] * gt[0] + sy[k] * gt[1]);                 // cotangent of the rotor thrust f_k
    const float gmk = sz[k] * gt[2];                                                  // ... of the rotor drag torque m_k
    const float aO = a_Om[k] + sd[k] * gdS;                                           // ... of dOm_k
    g_Om[k] += gfk * (pl.kf1 + 2.0f * pl.kf2 * Om[k]) + gmk * (pl.km1 + 2.0f * pl.km2 * Om[k]) + sd[k] * gS
             - aO * (cvk[k] + 2.0f * cdk[k] * Om[k]);                                 // Eq. (6)
    gu[k] += aO * (cvk[k] + 2.0f * cdk[k] * u[k]);
  }
  g_w[1] += pl.cJ[0] * w[2] * a_w[0]; g_w[2] += pl.cJ[0] * w[1] * a_w[0];
  g_w[2] += pl.cJ[1] * w[0] * a_w[1]; g_w[0] += pl.cJ[1] * w[2] * a_w[1];
  g_w[0] += pl.cJ[2] * w[1] * a_w[2]; g_w[1] += pl.cJ[2] * w[0] * a_w[2];
  // Eq. (2): dq = 1/2 q (x) (w, 0)
  float bx = 0.5f * a_q[0], by = 0.5f * a_q[1], bz = 0.5f * a_q[2], bw = 0.5f * a_q[3];
  g_q[3] += w[0] * bx + w[1] * by + w[2] * bz;
  g_q[0] += -w[2] * by + w[1] * bz - w[0] * bw;
  g_q[1] += w[2] * bx - w[0] * bz - w[1] * bw;
  g_q[2] += -w[1] * bx + w[0] * by - w[2] * bw;
  g_w[0] += q[3] * bx + q[2] * by - q[1] * bz - q[0] * bw;
  g_w[1] += -q[2] * bx + q[3] * by + q[0] * bz - q[1] * bw;
  g_w[2] += q[1] * bx - q[0] * by + q[3] * bz - q[2] * bw;
}

// ---- VJP of the abstracted derivative with the extras (deriv_ab<OPT_EXTRAS>): body drag, simplified model of
// PAPER.md:L354 (ab_thrust_dyn = 0: the thrust command acts directly, f_Sigma has no dynamics)
__device__ __forceinline__ void vjp_deriv_ab_ex(const DevParams &P, const Plant<MODEL_AB, GOPT> &pl, const float *x,
                                                const float *u, const float *a, float *gx, float *gu) {
  float sn[3], cs[3];
  sincos3_step(x + 3, sn, cs);
  const float sr = sn[0], cr = cs[0], sp = sn[1], cp = cs[1], sy = sn[2], cy = cs[2];
  const float *a_p = a, *a_ps = a + 3, *a_v = a + 6, *a_dps = a + 9;
  const float a_f = a[12];
  const bool simple = !P.ab_thrust_dyn;
  float zx = cy * sp * cr + sy * sr, zy = sy * sp * cr - cy * sr, zz = cp * cr;
  float acc = (P.ab_cf * (simple ? u[3] : x[12])) * pl.inv_m;
#pragma unroll
  for (int j = 0; j < 3; ++j) {
    gx[6 + j] += a_p[j];
    gx[9 + j] += a_ps[j] + pl.b[j] * a_dps[j];
    gx[3 + j] += pl.a[j] * a_dps[j];
    gu[j] += pl.c[j] * a_dps[j];
  }
  float dzr[3] = { -cy * sp * sr + sy * cr, -sy * sp * sr - cy * cr, -cp * sr };
  float dzp[3] = { cy * cp * cr, sy * cp * cr, -sp * cr };
  float dzy[3] = { -sy * sp * cr + cy * sr, cy * sp * cr + sy * sr, 0.0f };
  gx[3] += (dzr[0] * a_v[0] + dzr[1] * a_v[1] + dzr[2] * a_v[2]) * acc;
  gx[4] += (dzp[0] * a_v[0] + dzp[1] * a_v[1] + dzp[2] * a_v[2]) * acc;
  gx[5] += (dzy[0] * a_v[0] + dzy[1] * a_v[1]) * acc;
  const float g_fS = (zx * a_v[0] + zy * a_v[1] + zz * a_v[2]) * (P.ab_cf * pl.inv_m);
  if (simple) {
    gu[3] += g_fS;
  } else {
    gx[12] += g_fS - pl.ctau * a_f;                                                   // Eq. (9)
    gu[3] += pl.ctau * a_f;
  }
  if (P.has_drag) {
    float R[3][3], GR[3][3];
    euler_R_from_sc(sn, cs, R);
    vjp_drag(P, pl.inv_m, R, x + 6, a_v, gx + 6, GR);
    vjp_euler_R(R, sn, cs, GR, gx + 3);
  }
}

template <int MODEL, int OPT>
__device__ __forceinline__ void vjp_deriv(const DevParams &P, const Plant<MODEL, OPT> &pl, const float *x, const float *u,
                                          const float *a, float *gx, float *gu) {
  if constexpr (OPT != 0) {
    if constexpr (MODEL == MODEL_FP) vjp_deriv_fp_ex(P, pl, x, u, a, gx, gu);
    else vjp_deriv_ab_ex(P, pl, x, u, a, gx, gu);
  } else {
    if constexpr (MODEL == MODEL_FP) vjp_deriv_fp(P, pl, x, a, gx, gu);
    else vjp_deriv_ab(P, pl, x, a, gx, gu);
  }
}

// C6 motor mixer: (F_c, tau) -> rotor command.  Cotangent g_rpm[4] -> g_Fc (accumulated), g_tau[3] (assigned).  The
// forward pass is recomputed to know which clips are active (R33: derivative 0 there).  With a thrust polynomial
// (OPT_EXTRAS) r = (sqrt(kf1^2 - 4 kf2 (kf0 - f)) - kf1) / (2 kf2), so dr/df = 1 / sqrt(disc).
template <int OPT>
__device__ __forceinline__ void vjp_mixer(const DevParams &P, float Fc, const float *tau, const float *g_rpm, float *g_Fc,
                                          float *g_tau) {
  float a = 0.25f * Fc, bx = tau[0] * P.inv_4lever, by = tau[1] * P.inv_4lever, bz = tau[2] * P.inv_4kappa;
  float f[4] = { a - bx - by - bz, a - bx + by + bz, a + bx + by - bz, a + bx - by + bz };
  float gf[4];
#pragma unroll
  for (int k = 0; k < 4; ++k) {
    float fk = clipf(f[k], 0.0f, P.f_rotor_max);
    float r, drdf;
    bool ok = true;
    if ((OPT & OPT_EXTRAS) && P.thrust_poly) {
      float disc = P.kf[1] * P.kf[1] - 4.0f * P.kf[2] * (P.kf[0] - fk);
      ok = disc > 0.0f;
      float sd = sqrtf(fmaxf(disc, 0.0f));
      r = (sd - P.kf[1]) * (0.5f * P.inv_kf2);
      drdf = 1.0f / sd;
    } else {
      r = sqrtf(fk * P.inv_kf2);
      drdf = 0.5f * P.inv_kf2 / r;                                                          // d sqrt(f/kf)/df = 1/(2 kf r)
    }
    bool live = ok && f[k] > 0.0f && f[k] < P.f_rotor_max && r > P.rpm_min && r < P.rpm_max;   // R33: 0 where a clip is active
    gf[k] = live ? g_rpm[k] * drdf : 0.0f;
  }
  float g_a = (gf[0] + gf[1]) + (gf[2] + gf[3]);
  float g_bx = (gf[2] + gf[3]) - (gf[0] + gf[1]);
  float g_by = (gf[1] + gf[2]) - (gf[0] + gf[3]);
  float g_bz = (gf[1] + gf[3]) - (gf[0] + gf[2]);
  *g_Fc += 0.25f * g_a;
  g_tau[0] = g_bx * P.inv_4lever; g_tau[1] = g_by * P.inv_4lever; g_tau[2] = g_bz * P.inv_4kappa;
}

// ---- VJP of the attitude controller tick + mixer (C5, C6) -----------------------------------------------------------
// inputs of the tick: q, w (state), cmd = (roll, pitch, yaw, F), iR (integral before the tick).
// cotangents in: g_rpm[4] (of the rotor command), g_iRn[3] (of the integral after the tick).
// out: accumulates into g_q[4], g_w[3], g_cmd[4]; g_iR[3] = cotangent of the integral before the tick.
template <int OPT>
__device__ __forceinline__ void vjp_attitude_tick(const DevParams &P, const float *q, const float *w, const float *cmd,
                                                  const float *iR, const float *g_rpm, const float *g_iRn,
                                                  float *g_q, float *g_w, float *g_cmd, float *g_iR) {
  float R[3][3], Rd[3][3];
  quat_to_R(q, R);
  float sn[3], cs[3];                                             // one evaluation serves Rd and its angle derivatives;
  sincos3_step(cmd, sn, cs);                                      // MUFU (abs err 5e-7): a linearisation point, not the forward value
  euler_R_from_sc(sn, cs, Rd);
  auto Mij = [&](int i, int j) { return Rd[0][i] * R[0][j] + Rd[1][i] * R[1][j] + Rd[2][i] * R[2][j]; };
  float eR[3] = { 0.5f * (Mij(2, 1) - Mij(1, 2)), 0.5f * (Mij(0, 2) - Mij(2, 0)), 0.5f * (Mij(1, 0) - Mij(0, 1)) };
  float pre[3], iRn[3], tau[3];
#pragma unroll
  for (int j = 0; j < 3; ++j) {
    pre[j] = fmaf(eR[j], P.h_att, iR[j]);
    iRn[j] = clipf(pre[j], -P.iR_max, P.iR_max);
    tau[j] = P.Jnom[j] * (-P.kR[j] * eR[j] - P.kW[j] * w[j] - P.kI[j] * iRn[j]);
  }
  float g_tau[3];
  vjp_mixer<OPT>(P, cmd[3], tau, g_rpm, &g_cmd[3], g_tau);
  float g_eR[3];
#pragma unroll
  for (int j = 0; j < 3; ++j) {
    float gt = P.Jnom[j] * g_tau[j];
    g_eR[j] = -P.kR[j] * gt;
    g_w[j] += -P.kW[j] * gt;
    float g_in = g_iRn[j] - P.kI[j] * gt;                          // cotangent of the integral after the tick
    float g_pre = (pre[j] > -P.iR_max && pre[j] < P.iR_max) ? g_in : 0.0f;
    g_iR[j] = g_pre;
    g_eR[j] += P.h_att * g_pre;
  }
  // e_R = 1/2 (M21 - M12, M02 - M20, M10 - M01),  M = Rd^T R
  float G[3][3] = { { 0.0f, -0.5f * g_eR[2], 0.5f * g_eR[1] },
                    { 0.5f * g_eR[2], 0.0f, -0.5f * g_eR[0] },
                    { -0.5f * g_eR[1], 0.5f * g_eR[0], 0.0f } };        // G[i][j] = dL/dM_ij
  float GR[3][3], GD[3][3];
#pragma unroll
  for (int k = 0; k < 3; ++k)
#pragma unroll
    for (int j = 0; j < 3; ++j) {
      GR[k][j] = Rd[k][0] * G[0][j] + Rd[k][1] * G[1][j] + Rd[k][2] * G[2][j];     // dL/dR_kj
      GD[k][j] = R[k][0] * G[j][0] + R[k][1] * G[j][1] + R[k][2] * G[j][2];        // dL/dRd_kj
    }
  vjp_quat_to_R(q, GR, g_q);
  vjp_euler_R(Rd, sn, cs, GD, g_cmd);
}

// ---- one step forward (C4) from x with the inputs held: the rollout kernel's own integrator (lean first-principles
// step / generic Euler and RK4; quaternion renormalised; simplified abstracted model: f_Sigma <- f_cmd) ----------------
template <int MODEL, int INTEG, int OPT>
__device__ __forceinline__ void step_forward(const DevParams &P, const Plant<MODEL, OPT> &pl, float *x, const float *u,
                                             const float *fd) {
  constexpr int D = Dim<MODEL>::D;
  if constexpr (MODEL == MODEL_FP || OPT != 0) {
    integrate<MODEL, INTEG, OPT>(P, pl, x, u, fd);
    return;
  }
  float k[D];
  if constexpr (INTEG == INTEG_EULER) {
    deriv<MODEL, OPT>(P, pl, x, u, fd, k);
#pragma unroll
    for (int j = 0; j < D; ++j) x[j] = fmaf(P.h, k[j], x[j]);
  } else {
    float xs[D], acc[D];
    deriv<MODEL, OPT>(P, pl, x, u, fd, k);
#pragma unroll
    for (int j = 0; j < D; ++j) { acc[j] = k[j]; xs[j] = fmaf(P.half_h, k[j], x[j]); }
    deriv<MODEL, OPT>(P, pl, xs, u, fd, k);
#pragma unroll
    for (int j = 0; j < D; ++j) { acc[j] = fmaf(2.0f, k[j], acc[j]); xs[j] = fmaf(P.half_h, k[j], x[j]); }
    deriv<MODEL, OPT>(P, pl, xs, u, fd, k);
#pragma unroll
    for (int j = 0; j < D; ++j) { acc[j] = fmaf(2.0f, k[j], acc[j]); xs[j] = fmaf(P.h, k[j], x[j]); }
    deriv<MODEL, OPT>(P, pl, xs, u, fd, k);
#pragma unroll
    for (int j = 0; j < D; ++j) x[j] = fmaf(P.h_sixth, acc[j] + k[j], x[j]);
  }
}

// ---- pull the cotangent lam (of the post-step state) back through one step that started at x with held inputs u -----
// on return lam = cotangent of x, gu accumulates the cotangent of u.  fd: the step's disturbance force (held over the
// stages; it shifts the stage velocities, which the drag term reads)
template <int MODEL, int INTEG, int OPT>
__device__ __forceinline__ void step_backward(const DevParams &P, const Plant<MODEL, OPT> &pl, const float *x,
                                              const float *u, const float *fd, float *lam, float *gu) {
  constexpr int D = Dim<MODEL>::D;
  if constexpr (MODEL == MODEL_AB && OPT != 0) {
    if (!P.ab_thrust_dyn) { gu[3] += lam[12]; lam[12] = 0.0f; }                // simplified model: f_Sigma+ = f_cmd
  }
  float k1[D], x2[D], x3[D], x4[D], kk[D];
  deriv<MODEL, OPT>(P, pl, x, u, fd, k1);
  if constexpr (INTEG == INTEG_RK4) {
#pragma unroll
    for (int j = 0; j < D; ++j) x2[j] = fmaf(P.half_h, k1[j], x[j]);
    deriv<MODEL, OPT>(P, pl, x2, u, fd, kk);
#pragma unroll
    for (int j = 0; j < D; ++j) { k1[j] = fmaf(2.0f, kk[j], k1[j]); x3[j] = fmaf(P.half_h, kk[j], x[j]); }
    deriv<MODEL, OPT>(P, pl, x3, u, fd, kk);
#pragma unroll
    for (int j = 0; j < D; ++j) { k1[j] = fmaf(2.0f, kk[j], k1[j]); x4[j] = fmaf(P.h, kk[j], x[j]); }
  }
  if constexpr (MODEL == MODEL_FP) {
    // q+ = qt / |qt| with qt the integrator's un-normalised quaternion: g_qt = (g - q+ (q+ . g)) / |qt|
    float qt[4];
    if constexpr (INTEG == INTEG_RK4) {
      deriv<MODEL, OPT>(P, pl, x4, u, fd, kk);
#pragma unroll
      for (int j = 0; j < 4; ++j) qt[j] = fmaf(P.h_sixth, k1[3 + j] + kk[3 + j], x[3 + j]);
    } else {
#pragma unroll
      for (int j = 0; j < 4; ++j) qt[j] = fmaf(P.h, k1[3 + j], x[3 + j]);
    }
    float inv = rsqrtf(qt[0] * qt[0] + qt[1] * qt[1] + qt[2] * qt[2] + qt[3] * qt[3]);
    float dot = 0.f;
#pragma unroll
    for (int j = 0; j < 4; ++j) { qt[j] *= inv; dot = fmaf(qt[j], lam[3 + j], dot); }
#pragma unroll
    for (int j = 0; j < 4; ++j) lam[3 + j] = (lam[3 + j] - qt[j] * dot) * inv;
  }
  float a[D], gx[D];
  if constexpr (INTEG == INTEG_EULER) {
#pragma unroll
    for (int j = 0; j < D; ++j) { a[j] = P.h * lam[j]; gx[j] = 0.f; }
    vjp_deriv<MODEL, OPT>(P, pl, x, u, a, gx, gu);
#pragma unroll
    for (int j = 0; j < D; ++j) lam[j] += gx[j];
  } else {
    // x+ = x + h/6 (k1 + 2 k2 + 2 k3 + k4), k2 = f(x + h/2 k1), k3 = f(x + h/2 k2), k4 = f(x + h k3)
    float tot[D];
#pragma unroll
    for (int j = 0; j < D; ++j) { a[j] = P.h_sixth * lam[j]; gx[j] = 0.f; tot[j] = 0.f; }
    vjp_deriv<MODEL, OPT>(P, pl, x4, u, a, gx, gu);                           // k4
#pragma unroll
    for (int j = 0; j < D; ++j) { tot[j] += gx[j]; a[j] = fmaf(P.h, gx[j], 2.0f * P.h_sixth * lam[j]); gx[j] = 0.f; }
    vjp_deriv<MODEL, OPT>(P, pl, x3, u, a, gx, gu);                           // k3
#pragma unroll
    for (int j = 0; j < D; ++j) { tot[j] += gx[j]; a[j] = fmaf(P.half_h, gx[j], 2.0f * P.h_sixth * lam[j]); gx[j] = 0.f; }
    vjp_deriv<MODEL, OPT>(P, pl, x2, u, a, gx, gu);                           // k2
#pragma unroll
    for (int j = 0; j < D; ++j) { tot[j] += gx[j]; a[j] = fmaf(P.half_h, gx[j], P.h_sixth * lam[j]); gx[j] = 0.f; }
    vjp_deriv<MODEL, OPT>(P, pl, x, u, a, gx, gu);                            // k1
#pragma unroll
    for (int j = 0; j < D; ++j) lam[j] += tot[j] + gx[j];
  }
}

// ---- lean adjoint of the first-principles step (the exact transpose of integrate_fp_lean) -----------------------------
// The forward sweep runs the rollout kernel's lean step: stage states exist only for (q, w, Omega) -- position and
// velocity are carried in closed form, p+ = p + h v + h^2/6 (a1 + a2 + a3), v+ = v + h/6 (a1 + 2 a2 + 2 a3 + a4), and the
// rotor stages are Omega_i = u + e c_i with e = Omega - u.  Its transpose therefore needs, per stage, only the (dw, dq)
// part of the rates for the recomputation and ONE 10-cotangent VJP of fp_lean_rates (a(3), dw(3), dq(4) -> q, w, Omega);
// the cotangents of the accelerations come straight from (lam_p, lam_v) and feed nothing else.  Against the generic
// 17-component pull-back (4 deriv_fp + 4 vjp_deriv_fp + 17-wide RK4 bookkeeping) this is less than half the instructions.
__device__ __forceinline__ void fp_lean_dwdq(const Plant<MODEL_FP, 0> &pl, const float *q, const float *w, const float *Om,
                                             float *dw, float *dq) {
  float w2[4];
#pragma unroll
  for (int k = 0; k < 4; ++k) w2[k] = Om[k] * Om[k];
  const float A = w2[0] + w2[1], B = w2[2] + w2[3], C = w2[1] + w2[2], Dd = w2[0] + w2[3];
  const float E = w2[1] + w2[3], G = w2[0] + w2[2];
  dw[0] = fmaf(pl.cJ[0], w[1] * w[2], pl.ct[0] * (B - A));
  dw[1] = fmaf(pl.cJ[1], w[2] * w[0], pl.ct[1] * (C - Dd));
  dw[2] = fmaf(pl.cJ[2], w[0] * w[1], pl.ct[2] * (E - G));
  dq[0] = fmaf(q[3], w[0], fmaf(q[1], w[2], -(q[2] * w[1])));
  dq[1] = fmaf(q[3], w[1], fmaf(q[2], w[0], -(q[0] * w[2])));
  dq[2] = fmaf(q[3], w[2], fmaf(q[0], w[1], -(q[1] * w[0])));
  dq[3] = -fmaf(q[0], w[0], fmaf(q[1], w[1], q[2] * w[2]));
}
__device__ __forceinline__ void fp_lean_dq(const float *q, const float *w, float *dq) {
  dq[0] = fmaf(q[3], w[0], fmaf(q[1], w[2], -(q[2] * w[1])));
  dq[1] = fmaf(q[3], w[1], fmaf(q[2], w[0], -(q[0] * w[2])));
  dq[2] = fmaf(q[3], w[2], fmaf(q[0], w[1], -(q[1] * w[0])));
  dq[3] = -fmaf(q[0], w[0], fmaf(q[1], w[1], q[2] * w[2]));
}
// cotangents (ga, gdw, gdq) of fp_lean_rates at (q, w, Om) -> cotangents gq, gw, gO of its inputs (assigned)
__device__ __forceinline__ void vjp_fp_lean_rates(const Plant<MODEL_FP, 0> &pl, const float *q, const float *w,
                                                  const float *Om, const float *ga, const float *gdw, const float *gdq,
                                                  float *gq, float *gw, float *gO) {
  // a = (zx, zy, 1/2 - zh) acc2 + fa,  acc2 = kfm2 sum Om^2,  zx = q0 q2 + q3 q1, zy = q1 q2 - q3 q0, zh = q0^2 + q1^2
  const float s2 = fmaf(Om[0], Om[0], Om[1] * Om[1]) + fmaf(Om[2], Om[2], Om[3] * Om[3]);
  const float acc2 = pl.kfm2 * s2;
  const float zx = fmaf(q[0], q[2], q[3] * q[1]), zy = fmaf(q[1], q[2], -(q[3] * q[0])), zh = fmaf(q[0], q[0], q[1] * q[1]);
  const float g_acc2 = fmaf(zx, ga[0], fmaf(zy, ga[1], (0.5f - zh) * ga[2]));
  const float gzx = acc2 * ga[0], gzy = acc2 * ga[1], gzh2 = -2.0f * acc2 * ga[2];
  // dw_j = cJ_j w_a w_b + ct_j (signed sum of Om^2): signs (B - A), (C - Dd), (E - G)
  const float t0 = pl.ct[0] * gdw[0], t1 = pl.ct[1] * gdw[1], t2 = pl.ct[2] * gdw[2];
  const float s = pl.kfm2 * g_acc2, sm = s - t0, sp = s + t0, u = t1 + t2, v = t1 - t2;
  gO[0] = 2.0f * Om[0] * (sm - u);
  gO[1] = 2.0f * Om[1] * (sm + u);
  gO[2] = 2.0f * Om[2] * (sp + v);
  gO[3] = 2.0f * Om[3] * (sp - v);
  const float c0 = pl.cJ[0] * gdw[0], c1 = pl.cJ[1] * gdw[1], c2 = pl.cJ[2] * gdw[2];
  // dq = 2 q-dot:  dq0 = q3 w0 + q1 w2 - q2 w1, dq1 = q3 w1 + q2 w0 - q0 w2, dq2 = q3 w2 + q0 w1 - q1 w0, dq3 = -(q . w)
  gw[0] = fmaf(w[2], c1, fmaf(w[1], c2, fmaf(q[3], gdq[0], fmaf(q[2], gdq[1], -fmaf(q[1], gdq[2], q[0] * gdq[3])))));
  gw[1] = fmaf(w[2], c0, fmaf(w[0], c2, fmaf(q[3], gdq[1], fmaf(q[0], gdq[2], -fmaf(q[2], gdq[0], q[1] * gdq[3])))));
  gw[2] = fmaf(w[1], c0, fmaf(w[0], c1, fmaf(q[3], gdq[2], fmaf(q[1], gdq[0], -fmaf(q[0], gdq[1], q[2] * gdq[3])))));
  gq[0] = fmaf(q[2], gzx, fmaf(q[0], gzh2, fmaf(w[1], gdq[2], -fmaf(q[3], gzy, fmaf(w[2], gdq[1], w[0] * gdq[3])))));
  gq[1] = fmaf(q[3], gzx, fmaf(q[2], gzy, fmaf(q[1], gzh2, fmaf(w[2], gdq[0], -fmaf(w[0], gdq[2], w[1] * gdq[3])))));
  gq[2] = fmaf(q[0], gzx, fmaf(q[1], gzy, fmaf(w[0], gdq[1], -fmaf(w[1], gdq[0], w[2] * gdq[3]))));
  gq[3] = fmaf(q[1], gzx, fmaf(w[0], gdq[0], fmaf(w[1], gdq[1], fmaf(w[2], gdq[2], -(q[0] * gzy)))));
}

// lam (cotangent of the post-step state, 17 components) -> cotangent of the pre-step state; gu accumulates the
// cotangent of the held rotor command u.  x: pre-step state, only q (3..6), w (10..12), Omega (13..16) are read.
template <int INTEG>
__device__ __forceinline__ void step_backward_fp_lean(const DevParams &P, const Plant<MODEL_FP, 0> &pl, const float *x,
                                                      const float *u, float *lam, float *gu) {
  const float *q = x + 3, *w = x + 10, *Om = x + 13;
  float *lp = lam, *lq = lam + 3, *lv = lam + 7, *lw = lam + 10, *lO = lam + 13;
  float e[4];
#pragma unroll
  for (int k = 0; k < 4; ++k) e[k] = Om[k] - u[k];
  const float hq = 0.5f * P.h;
  if constexpr (INTEG == INTEG_EULER) {
    float dq1[4], qt[4];
    fp_lean_dq(q, w, dq1);
#pragma unroll
    for (int j = 0; j < 4; ++j) qt[j] = fmaf(hq, dq1[j], q[j]);
    const float inv = rsqrtf(fmaf(qt[0], qt[0], fmaf(qt[1], qt[1], fmaf(qt[2], qt[2], qt[3] * qt[3]))));
    float dot = 0.f;
#pragma unroll
    for (int j = 0; j < 4; ++j) { qt[j] *= inv; dot = fmaf(qt[j], lq[j], dot); }
#pragma unroll
    for (int j = 0; j < 4; ++j) lq[j] = (lq[j] - qt[j] * dot) * inv;
    float ga[3], gdw[3], gdq[4], gq[4], gw[3], gO[4];
#pragma unroll
    for (int j = 0; j < 3; ++j) { ga[j] = P.h * lv[j]; gdw[j] = P.h * lw[j]; }
#pragma unroll
    for (int j = 0; j < 4; ++j) gdq[j] = hq * lq[j];
    vjp_fp_lean_rates(pl, q, w, Om, ga, gdw, gdq, gq, gw, gO);
#pragma unroll
    for (int j = 0; j < 3; ++j) { lv[j] = fmaf(P.h, lp[j], lv[j]); lw[j] += gw[j]; }
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      lq[j] += gq[j];
      const float ge = fmaf(pl.rho1, lO[j], gO[j]);
      gu[j] += (gO[j] + lO[j]) - ge;
      lO[j] = ge;
    }
  } else {
    float q2[4], q3[4], q4[4], w2[3], w3[3], w4[3], O2[4], O3[4], O4[4], dw[3], dq[4], qt[4];
    fp_lean_dwdq(pl, q, w, Om, dw, dq);
#pragma unroll
    for (int j = 0; j < 4; ++j) { qt[j] = dq[j]; q2[j] = fmaf(0.5f * hq, dq[j], q[j]); O2[j] = fmaf(e[j], pl.rc2, u[j]); }
#pragma unroll
    for (int j = 0; j < 3; ++j) w2[j] = fmaf(P.half_h, dw[j], w[j]);
    fp_lean_dwdq(pl, q2, w2, O2, dw, dq);
#pragma unroll
    for (int j = 0; j < 4; ++j) { qt[j] = fmaf(2.0f, dq[j], qt[j]); q3[j] = fmaf(0.5f * hq, dq[j], q[j]); O3[j] = fmaf(e[j], pl.rc3, u[j]); }
#pragma unroll
    for (int j = 0; j < 3; ++j) w3[j] = fmaf(P.half_h, dw[j], w[j]);
    fp_lean_dwdq(pl, q3, w3, O3, dw, dq);
#pragma unroll
    for (int j = 0; j < 4; ++j) { qt[j] = fmaf(2.0f, dq[j], qt[j]); q4[j] = fmaf(hq, dq[j], q[j]); O4[j] = fmaf(e[j], pl.rc4, u[j]); }
#pragma unroll
    for (int j = 0; j < 3; ++j) w4[j] = fmaf(P.h, dw[j], w[j]);
    fp_lean_dq(q4, w4, dq);
    const float hq6 = 0.5f * P.h_sixth, h2_6 = P.h * P.h_sixth;
#pragma unroll
    for (int j = 0; j < 4; ++j) qt[j] = fmaf(hq6, qt[j] + dq[j], q[j]);
    // q+ = qt / |qt|:  g_qt = (g - q+ (q+ . g)) / |qt|
    const float inv = rsqrtf(fmaf(qt[0], qt[0], fmaf(qt[1], qt[1], fmaf(qt[2], qt[2], qt[3] * qt[3]))));
    float dot = 0.f;
#pragma unroll
    for (int j = 0; j < 4; ++j) { qt[j] *= inv; dot = fmaf(qt[j], lq[j], dot); }
#pragma unroll
    for (int j = 0; j < 4; ++j) lq[j] = (lq[j] - qt[j] * dot) * inv;
    // stage cotangents, last stage first
    float gaA[3], gaB[3], gaC[3], lw6[3], lq6[4];
#pragma unroll
    for (int j = 0; j < 3; ++j) {
      gaC[j] = P.h_sixth * lv[j];
      const float hp = h2_6 * lp[j];
      gaA[j] = hp + gaC[j];
      gaB[j] = fmaf(2.0f, gaC[j], hp);
      lw6[j] = P.h_sixth * lw[j];
    }
#pragma unroll
    for (int j = 0; j < 4; ++j) lq6[j] = hq6 * lq[j];
    float gdw[3], gdq[4], gq[4], gw[3], gO[4], ge[4], gus[4];
    vjp_fp_lean_rates(pl, q4, w4, O4, gaC, lw6, lq6, gq, gw, gO);                     // k4
#pragma unroll
    for (int j = 0; j < 4; ++j) { ge[j] = pl.rc4 * gO[j]; gus[j] = gO[j]; lq[j] += gq[j]; gdq[j] = fmaf(hq, gq[j], 2.0f * lq6[j]); }
#pragma unroll
    for (int j = 0; j < 3; ++j) { lw[j] += gw[j]; gdw[j] = fmaf(P.h, gw[j], 2.0f * lw6[j]); }
    vjp_fp_lean_rates(pl, q3, w3, O3, gaB, gdw, gdq, gq, gw, gO);                     // k3
#pragma unroll
    for (int j = 0; j < 4; ++j) { ge[j] = fmaf(pl.rc3, gO[j], ge[j]); gus[j] += gO[j]; lq[j] += gq[j]; gdq[j] = fmaf(0.5f * hq, gq[j], 2.0f * lq6[j]); }
#pragma unroll
    for (int j = 0; j < 3; ++j) { lw[j] += gw[j]; gdw[j] = fmaf(P.half_h, gw[j], 2.0f * lw6[j]); }
    vjp_fp_lean_rates(pl, q2, w2, O2, gaB, gdw, gdq, gq, gw, gO);                     // k2
#pragma unroll
    for (int j = 0; j < 4; ++j) { ge[j] = fmaf(pl.rc2, gO[j], ge[j]); gus[j] += gO[j]; lq[j] += gq[j]; gdq[j] = fmaf(0.5f * hq, gq[j], lq6[j]); }
#pragma unroll
    for (int j = 0; j < 3; ++j) { lw[j] += gw[j]; gdw[j] = fmaf(P.half_h, gw[j], lw6[j]); }
    vjp_fp_lean_rates(pl, q, w, Om, gaA, gdw, gdq, gq, gw, gO);                       // k1
#pragma unroll
    for (int j = 0; j < 3; ++j) { lw[j] += gw[j]; lv[j] = fmaf(P.h, lp[j], lv[j]); }
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      lq[j] += gq[j];
      const float g_e = fmaf(pl.rho4, lO[j], ge[j] + gO[j]);
      gu[j] += (gus[j] + gO[j] + lO[j]) - g_e;
      lO[j] = g_e;
    }
  }
}

// ---- VJP of the geometric position controller tick (C7, reading R16) ----------------------------------------------------
// inputs of the tick: p, v (state), zB (body z axis in the world frame), target = (x, y, z, yaw), ip (integral before).
// cotangents in: g_att[4] of the attitude command (roll, pitch, yaw, F) the tick produced, g_ipn[3] of the integral
// after the tick.  out: accumulates into g_p[3], g_v[3], g_zB[3], g_tg[4]; g_ip[3] = cotangent of the integral before.
// Where a clip of the method is active (integral, thrust, tilt, asin argument, norm floors) the derivative is 0 (R33).
__device__ __forceinline__ void vjp_position_tick(const DevParams &P, const float *pos, const float *vel, const float *zB,
                                                  const float *target, const float *ip, const float *g_att,
                                                  const float *g_ipn, float *g_p, float *g_v, float *g_zB, float *g_tg,
                                                  float *g_ip) {
  // forward recomputation (same arithmetic as position_tick, accurate trigonometry: this is a linearisation point)
  float ep[3], pre[3], t[3];
#pragma unroll
  for (int j = 0; j < 3; ++j) {
    ep[j] = target[j] - pos[j];
    pre[j] = fmaf(ep[j], P.h_pos, ip[j]);
    float ipn = clipf(pre[j], -P.ip_max[j], P.ip_max[j]);
    float ad = P.kp[j] * ep[j] - P.kd[j] * vel[j] + P.ki[j] * ipn + (j == 2 ? P.g : 0.0f);
    t[j] = P.mass * ad;
  }
  const float Fraw = t[0] * zB[0] + t[1] * zB[1] + t[2] * zB[2];
  const float n2 = t[0] * t[0] + t[1] * t[1] + t[2] * t[2];
  const bool n_live = n2 > 1e-12f;
  const float inv = rsqrtf(fmaxf(n2, 1e-12f));
  const float zd[3] = { t[0] * inv, t[1] * inv, t[2] * inv };
  float sy, cy;
  sincosf(target[3], &sy, &cy);
  const float yr[3] = { -zd[2] * sy, zd[2] * cy, zd[0] * sy - zd[1] * cy };
  const float ny2 = yr[0] * yr[0] + yr[1] * yr[1] + yr[2] * yr[2];
  const bool y_live = ny2 > 1e-12f;
  const float invy = rsqrtf(fmaxf(ny2, 1e-12f));
  const float yd[3] = { yr[0] * invy, yr[1] * invy, yr[2] * invy };
  const float xd[3] = { yd[1] * zd[2] - yd[2] * zd[1], yd[2] * zd[0] - yd[0] * zd[2], yd[0] * zd[1] - yd[1] * zd[0] };
  const float roll_raw = atan2f(yd[2], zd[2]);
  const float sarg = -xd[2];
  const float pitch_raw = asinf(clipf(sarg, -1.0f, 1.0f));
  // reverse
  float g_xd[3] = { 0.f, 0.f, 0.f }, g_yd[3] = { 0.f, 0.f, 0.f }, g_zd[3] = { 0.f, 0.f, 0.f };
  {                                                   // yaw = atan2(xd_y, xd_x)
    const float r2 = xd[0] * xd[0] + xd[1] * xd[1];
    if (r2 > 0.f) { g_xd[1] += g_att[2] * xd[0] / r2; g_xd[0] -= g_att[2] * xd[1] / r2; }
  }
  if (fabsf(pitch_raw) < P.tilt_max && fabsf(sarg) < 1.0f)          // pitch = asin(-xd_z)
    g_xd[2] -= g_att[1] * rsqrtf(fmaxf(1.0f - sarg * sarg, 1e-20f));
  if (fabsf(roll_raw) < P.tilt_max) {                                 // roll = atan2(yd_z, zd_z)
    const float r2 = yd[2] * yd[2] + zd[2] * zd[2];
    if (r2 > 0.f) { g_yd[2] += g_att[0] * zd[2] / r2; g_zd[2] -= g_att[0] * yd[2] / r2; }
  }
  // xd = yd x zd:  g_yd += zd x g_xd,  g_zd += g_xd x yd
  g_yd[0] += zd[1] * g_xd[2] - zd[2] * g_xd[1]; g_yd[1] += zd[2] * g_xd[0] - zd[0] * g_xd[2]; g_yd[2] += zd[0] * g_xd[1] - zd[1] * g_xd[0];
  g_zd[0] += g_xd[1] * yd[2] - g_xd[2] * yd[1]; g_zd[1] += g_xd[2] * yd[0] - g_xd[0] * yd[2]; g_zd[2] += g_xd[0] * yd[1] - g_xd[1] * yd[0];
  // yd = yr / |yr|
  float g_yr[3];
  {
    const float dot = yd[0] * g_yd[0] + yd[1] * g_yd[1] + yd[2] * g_yd[2];
#pragma unroll
    for (int j = 0; j < 3; ++j) g_yr[j] = y_live ? invy * (g_yd[j] - yd[j] * dot) : invy * g_yd[j];
  }
  // yr = (-zd_z sy, zd_z cy, zd_x sy - zd_y cy)
  g_zd[2] += -sy * g_yr[0] + cy * g_yr[1];
  g_zd[0] += sy * g_yr[2];
  g_zd[1] -= cy * g_yr[2];
  g_tg[3] += g_yr[0] * (-zd[2] * cy) + g_yr[1] * (-zd[2] * sy) + g_yr[2] * (zd[0] * cy + zd[1] * sy);
  // zd = t / |t|
  float g_t[3];
  {
    const float dot = zd[0] * g_zd[0] + zd[1] * g_zd[1] + zd[2] * g_zd[2];
#pragma unroll
    for (int j = 0; j < 3; ++j) g_t[j] = n_live ? inv * (g_zd[j] - zd[j] * dot) : inv * g_zd[j];
  }
  // F = clip(t . zB)
  if (Fraw > P.thrust_min && Fraw < P.thrust_max) {
#pragma unroll
    for (int j = 0; j < 3; ++j) { g_t[j] += g_att[3] * zB[j]; g_zB[j] += g_att[3] * t[j]; }
  }
#pragma unroll
  for (int j = 0; j < 3; ++j) {
    const float g_ad = P.mass * g_t[j];
    float g_ep = P.kp[j] * g_ad;
    g_v[j] -= P.kd[j] * g_ad;
    const float g_in = g_ipn[j] + P.ki[j] * g_ad;
    const float g_pre = (pre[j] > -P.ip_max[j] && pre[j] < P.ip_max[j]) ? g_in : 0.0f;
    g_ip[j] = g_pre;
    g_ep += P.h_pos * g_pre;
    g_tg[j] += g_ep;
    g_p[j] -= g_ep;
  }
}

// body z axis in the world frame and the pull-back of its cotangent to the attitude state
__device__ __forceinline__ void zB_fp(const float *q, float *zB) {
  zB[0] = 2.0f * (q[0] * q[2] + q[3] * q[1]);
  zB[1] = 2.0f * (q[1] * q[2] - q[3] * q[0]);
  zB[2] = 1.0f - 2.0f * (q[0] * q[0] + q[1] * q[1]);
}
__device__ __forceinline__ void vjp_zB_fp(const float *q, const float *gz, float *g_q) {
  g_q[0] += 2.0f * (q[2] * gz[0] - q[3] * gz[1]) - 4.0f * q[0] * gz[2];
  g_q[1] += 2.0f * (q[3] * gz[0] + q[2] * gz[1]) - 4.0f * q[1] * gz[2];
  g_q[2] += 2.0f * (q[0] * gz[0] + q[1] * gz[1]);
  g_q[3] += 2.0f * (q[1] * gz[0] - q[0] * gz[1]);
}
__device__ __forceinline__ void zB_ab(const float *psi, float *zB, float *sn, float *cs) {
  sincos3_step(psi, sn, cs);
  zB[0] = cs[2] * sn[1] * cs[0] + sn[2] * sn[0]; zB[1] = sn[2] * sn[1] * cs[0] - cs[2] * sn[0]; zB[2] = cs[1] * cs[0];
}
__device__ __forceinline__ void vjp_zB_ab(const float *sn, const float *cs, const float *gz, float *g_psi) {
  const float sr = sn[0], cr = cs[0], sp = sn[1], cp = cs[1], sy = sn[2], cy = cs[2];
  g_psi[0] += (-cy * sp * sr + sy * cr) * gz[0] + (-sy * sp * sr - cy * cr) * gz[1] + (-cp * sr) * gz[2];
  g_psi[1] += (cy * cp * cr) * gz[0] + (sy * cp * cr) * gz[1] + (-sp * cr) * gz[2];
  g_psi[2] += (-sy * sp * cr + cy * sr) * gz[0] + (cy * sp * cr + sy * sr) * gz[1];
}

// History of one step: only what the backward sweep reads NON-linearly.  Position and velocity enter Eqs. (1)-(4) /
// (7)-(10) linearly (no drag here), so without the position controller they are neither parked nor re-read:
//   FP rotor     16 floats: q(4) w(3) - Omega(4) rotor command(4)
//   FP attitude  18 floats: q(4) w(3) iR_0 Omega(4) rotor command(4) | iR_1 iR_2        (4 float4 + 1 float2)
//   FP position  32 floats: the 17 state floats, iR(3), ip(3), rotor command(4), attitude command after the tick(4), pad
//   AB attitude   8 floats: Psi(3) dPsi(3) f_Sigma pad
//   AB position  20 floats: the 13 state floats, ip(3), attitude command after the tick(4)
// Layout: all float4 planes first, [n_steps][H4][MN] float4, then the float2 planes [n_steps][MN] (FP attitude only), so
// every plane is aligned whatever MN is; a warp writes 512 (256) contiguous bytes per plane.
#ifndef GRAD_MIN_BLOCKS
#define GRAD_MIN_BLOCKS 4
#endif
template <int MODEL, int IFACE, int OPT = 0> struct Hist {
  static constexpr bool POS = IFACE == IF_POSITION || OPT != 0;     // general kernels park the full record
  static constexpr int HD = MODEL == MODEL_FP ? (POS ? 32 : (IFACE == IF_ATTITUDE ? 18 : 16)) : (POS ? 20 : 8);
  static constexpr int H4 = HD / 4, H2 = (HD % 4) / 2;
};

// Two launches per cf_grad call: PHASE 1 = forward sweep (parks the history, the loss and its cotangent), PHASE 2 =
// backward sweep.  As ONE kernel the two loop bodies (12 KB + 29 KB of code) are live on an SM at the same time --
// blocks of different waves are in different sweeps -- and "no instruction" was the largest stall; split, each launch's
// loop fits the instruction cache on its own: 0.793 -> 0.761 ms for 2^20 worlds x 10 RK4 steps (same GPU).  Launch bounds
// 3 / 5 / 6 / 8 blocks for either phase measured no better than 4.
// General kernels (OPT = GOPT: fidelity extras gated at run time by the DevParams flags, disturbances, torque interface):
// the generic integrator and 17 / 13-wide pull-back, full record per step, 2 blocks per SM (<= 255 registers).
template <int MODEL, int INTEG, int IFACE, int PHASE, int OPT = 0>
__global__ void __launch_bounds__(128, OPT != 0 ? 2 : GRAD_MIN_BLOCKS)
grad_kernel(const __grid_constant__ GradArgs A, const __grid_constant__ DevParams P, int randp) {
  using H = Hist<MODEL, IFACE, OPT>;
  constexpr bool GEN = OPT != 0;
  constexpr bool FULL = H::POS;
  constexpr int D = Dim<MODEL>::D, HD = H::HD, H4 = H::H4, HP = H4 * 4 + 4;
  constexpr bool FP = MODEL == MODEL_FP;
  constexpr bool POS = IFACE == IF_POSITION;
  constexpr bool HAS_ATT = FP && IFACE >= IF_ATTITUDE;
  constexpr int VEL = FP ? 7 : 6;
  const long long MN = A.MN;
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= MN) return;
  Plant<MODEL, OPT> pl;
  const long long w_loc = i / A.N;
  pl.load(P, A.wparam, A.M, w_loc, randp != 0);
  // C8 step 4: the disturbance of step s is sigma (z0, z1, z2) from Philox(seed; global world, drone, s, DIST)
  const uint32_t wg = (uint32_t)(w_loc + A.world_offset), nn = (uint32_t)(i - w_loc * A.N);
  auto disturbance = [&](uint32_t step, float *fd) {
    fd[0] = fd[1] = fd[2] = 0.0f;
    if constexpr (GEN) {
      if (P.dist_sigma > 0.0f) {
        uint32_t r[4]; float z[4];
        philox4x32_10_rk(A.rk, wg, nn, step, STREAM_DIST, r);
        normal_pair(r[0], r[1], z[0], z[1]);
        normal_pair(r[2], r[3], z[2], z[3]);
#pragma unroll
        for (int j = 0; j < 3; ++j) fd[j] = P.dist_sigma * z[j];
      }
    }
  };

  float x[D], iR[3] = { 0, 0, 0 }, ip[3] = { 0, 0, 0 }, rpm_cmd[4] = { 0, 0, 0, 0 }, cmd[4] = { 0, 0, 0, 0 };
  float att_cmd[4] = { 0, 0, 0, 0 };      // position interface: the attitude command the outer loop holds
#pragma unroll
  for (int j = 0; j < D; ++j) x[j] = A.state[j * MN + i];
  if (FP) {
#pragma unroll
    for (int j = 0; j < 3; ++j) iR[j] = A.ctrl[j * MN + i];
#pragma unroll
    for (int j = 0; j < 4; ++j) rpm_cmd[j] = A.ctrl[(10 + j) * MN + i];
  }
  if (FULL) {
#pragma unroll
    for (int j = 0; j < 3; ++j) ip[j] = A.ctrl[(3 + j) * MN + i];
#pragma unroll
    for (int j = 0; j < 4; ++j) att_cmd[j] = A.ctrl[(6 + j) * MN + i];
  }
  float4 *const h4 = A.hist;
  float2 *const h2 = reinterpret_cast<float2 *>(A.hist + (size_t)A.n_steps * H4 * MN);
  // pack / unpack of one step's record (see the table above)
  auto pack = [&](float *rec) {
#pragma unroll
    for (int j = 0; j < HP; ++j) rec[j] = 0.f;
    if constexpr (FULL) {
#pragma unroll
      for (int j = 0; j < D; ++j) rec[j] = x[j];
      int o = D;
      if (FP) {
#pragma unroll
        for (int j = 0; j < 3; ++j) rec[o + j] = iR[j];
        o += 3;
      }
#pragma unroll
      for (int j = 0; j < 3; ++j) rec[o + j] = ip[j];
    } else if constexpr (FP) {
#pragma unroll
      for (int j = 0; j < 4; ++j) { rec[j] = x[3 + j]; rec[8 + j] = x[13 + j]; }
#pragma unroll
      for (int j = 0; j < 3; ++j) rec[4 + j] = x[10 + j];
      if (HAS_ATT) { rec[7] = iR[0]; rec[16] = iR[1]; rec[17] = iR[2]; }
    } else {
#pragma unroll
      for (int j = 0; j < 3; ++j) { rec[j] = x[3 + j]; rec[3 + j] = x[9 + j]; }
      rec[6] = x[12];
    }
  };
  // ---- forward sweep -----------------------------------------------------------------------------------------
  int att_phase = (int)(A.s0 % (uint32_t)P.att_div), pos_phase = (int)(A.s0 % (uint32_t)P.pos_div);
  float4 *const lam0 = A.hist + ((size_t)A.n_steps * HD * MN + 3) / 4;       // [MN] float4 after the history (split launches)
  // Commands are prefetched one command ahead into registers by an UNCONDITIONAL load (index clamped to the last command:
  // a harmless re-load): a load behind the fetch test is not issued ahead by the compiler (the same change took the
  // rollout kernel's command-buffer loop from 0.495 to 0.361 ms)
  float4 c_next = make_float4(0.f, 0.f, 0.f, 0.f);
  if constexpr (PHASE != 2) c_next = __ldg(A.cmds + i);
  if constexpr (PHASE != 2)
  for (int t = 0, hold_phase = 0, k_cmd = 0; t < A.n_steps; ++t) {      // t = k_cmd * cmd_hold + hold_phase, no division
    float rec[HP];                                          // pre-step state and controller state of this step
    pack(rec);
    const float4 c4 = c_next;
    c_next = __ldg(A.cmds + (size_t)(k_cmd + 1 < A.n_cmds ? k_cmd + 1 : k_cmd) * MN + i);
    if (hold_phase == 0) {
      cmd[0] = c4.x; cmd[1] = c4.y; cmd[2] = c4.z; cmd[3] = c4.w;
      if (FP && IFACE == IF_ROTOR) {
#pragma unroll
        for (int j = 0; j < 4; ++j) rpm_cmd[j] = clipf(cmd[j], P.rpm_min, P.rpm_max);
      }
      if (FP && IFACE == IF_TORQUE) mixer<OPT>(P, cmd[3], cmd, rpm_cmd);      // (tau_x, tau_y, tau_z, F) straight into the mixer
    }
    if (++hold_phase == A.cmd_hold) { hold_phase = 0; ++k_cmd; }
    if (POS) {
      if (pos_phase == 0) {
        float zB[3], sn[3], cs[3];
        if (FP) zB_fp(x + 3, zB); else zB_ab(x + 3, zB, sn, cs);
        position_tick(P, x, x + VEL, zB, cmd, ip, att_cmd);
      }
      pos_phase = pos_phase + 1 == P.pos_div ? 0 : pos_phase + 1;
    }
    const float *acmd = POS ? att_cmd : cmd;                // the attitude command in force at this step
    if (HAS_ATT) {
      if (att_phase == 0) {
        float Rd[3][3];
        euler_to_R(acmd[0], acmd[1], acmd[2], Rd);
        attitude_tick<OPT>(P, x + 3, x + 10, Rd, acmd[3], iR, rpm_cmd);
      }
      att_phase = att_phase + 1 == P.att_div ? 0 : att_phase + 1;
    }
    if constexpr (FULL) {
      constexpr int o = FP ? D + 6 : D + 3;
      if (FP) {
#pragma unroll
        for (int j = 0; j < 4; ++j) rec[o + j] = rpm_cmd[j];
      }
#pragma unroll
      for (int j = 0; j < 4; ++j) rec[o + (FP ? 4 : 0) + j] = att_cmd[j];
    } else if constexpr (FP) {
#pragma unroll
      for (int j = 0; j < 4; ++j) rec[12 + j] = rpm_cmd[j];
    }
#pragma unroll
    for (int j = 0; j < H4; ++j)
      __stcs(h4 + ((size_t)t * H4 + j) * MN + i, make_float4(rec[4 * j], rec[4 * j + 1], rec[4 * j + 2], rec[4 * j + 3]));
    if constexpr (H::H2) __stcs(h2 + (size_t)t * MN + i, make_float2(rec[4 * H4], rec[4 * H4 + 1]));
    float fd[3];
    disturbance(A.s0 + (uint32_t)t, fd);
    step_forward<MODEL, INTEG, OPT>(P, pl, x, FP ? rpm_cmd : acmd, fd);
  }
  // ---- loss and its cotangent ----------------------------------------------------------------------------------
  float lam[D];
#pragma unroll
  for (int j = 0; j < D; ++j) lam[j] = 0.f;
  if constexpr (PHASE != 2) {
    float ex = x[0] - A.goal[0], ey = x[1] - A.goal[1], ez = x[2] - A.goal[2];
    float L = sqrtf(ex * ex + ey * ey + ez * ez);
    A.loss[i] = L;
    float inv = L > 0.f ? 1.0f / L : 0.f;
    lam[0] = ex * inv; lam[1] = ey * inv; lam[2] = ez * inv;
    if constexpr (PHASE == 1) { lam0[i] = make_float4(lam[0], lam[1], lam[2], 0.f); return; }
  } else {
    const float4 l4 = lam0[i];
    lam[0] = l4.x; lam[1] = l4.y; lam[2] = l4.z;
  }
  // ---- backward sweep ------------------------------------------------------------------------------------------
  float g_cmd[4] = { 0, 0, 0, 0 };      // cotangent of the held command, until its fetch step is reached
  float g_rpm[4] = { 0, 0, 0, 0 };      // cotangent of the held rotor command, until the tick / fetch that set it
  float g_iR[3] = { 0, 0, 0 };          // cotangent of the attitude controller's integral
  float g_att[4] = { 0, 0, 0, 0 };      // position interface: cotangent of the held attitude command, until the tick that set it
  float g_ip[3] = { 0, 0, 0 };          // cotangent of the position controller's integral
  att_phase = (int)((A.s0 + (uint32_t)A.n_steps - 1u) % (uint32_t)P.att_div);
  pos_phase = (int)((A.s0 + (uint32_t)A.n_steps - 1u) % (uint32_t)P.pos_div);
#pragma unroll
  for (int j = 0; j < D; ++j) x[j] = 0.f;                   // components that are not parked enter only linearly
  int hold_phase = (A.n_steps - 1) % A.cmd_hold, k_cmd = (A.n_steps - 1) / A.cmd_hold;    // of step t, kept by counting
  for (int t = A.n_steps - 1; t >= 0; --t) {
    float rec[HP];
    if (t > 0) {            // pull the previous step's record towards L2 while this step's pull-back computes
#pragma unroll
      for (int j = 0; j < H4; ++j) asm volatile("prefetch.global.L2 [%0];" :: "l"(h4 + ((size_t)(t - 1) * H4 + j) * MN + i));
      if constexpr (H::H2) asm volatile("prefetch.global.L2 [%0];" :: "l"(h2 + (size_t)(t - 1) * MN + i));
    }
#pragma unroll
    for (int j = 0; j < H4; ++j) {
      const float4 v = __ldcs(h4 + ((size_t)t * H4 + j) * MN + i);
      rec[4 * j] = v.x; rec[4 * j + 1] = v.y; rec[4 * j + 2] = v.z; rec[4 * j + 3] = v.w;
    }
    if constexpr (H::H2) { const float2 v = __ldcs(h2 + (size_t)t * MN + i); rec[4 * H4] = v.x; rec[4 * H4 + 1] = v.y; }
    if constexpr (FULL) {
#pragma unroll
      for (int j = 0; j < D; ++j) x[j] = rec[j];
      int o = D;
      if (FP) {
#pragma unroll
        for (int j = 0; j < 3; ++j) iR[j] = rec[o + j];
        o += 3;
      }
#pragma unroll
      for (int j = 0; j < 3; ++j) ip[j] = rec[o + j];
      o += 3;
      if (FP) {
#pragma unroll
        for (int j = 0; j < 4; ++j) rpm_cmd[j] = rec[o + j];
        o += 4;
      }
#pragma unroll
      for (int j = 0; j < 4; ++j) att_cmd[j] = rec[o + j];
    } else if constexpr (FP) {
#pragma unroll
      for (int j = 0; j < 4; ++j) { x[3 + j] = rec[j]; x[13 + j] = rec[8 + j]; rpm_cmd[j] = rec[12 + j]; }
#pragma unroll
      for (int j = 0; j < 3; ++j) x[10 + j] = rec[4 + j];
      if (HAS_ATT) { iR[0] = rec[7]; iR[1] = rec[16]; iR[2] = rec[17]; }
    } else {
#pragma unroll
      for (int j = 0; j < 3; ++j) { x[3 + j] = rec[j]; x[9 + j] = rec[3 + j]; }
      x[12] = rec[6];
    }
    if (hold_phase == A.cmd_hold - 1 || t == A.n_steps - 1) {                 // entering the run of command k_cmd
      float4 c4 = __ldg(A.cmds + (size_t)k_cmd * MN + i);
      cmd[0] = c4.x; cmd[1] = c4.y; cmd[2] = c4.z; cmd[3] = c4.w;
    }
    const float *acmd = POS ? att_cmd : cmd;
    float *g_acmd = POS ? g_att : g_cmd;
    // (tried and rejected, measured: the four RK4 stages of this pull-back rolled into run-time loops with the stage
    //  states in shared memory -- "no instruction" stalls 1.03 -> 0.13 per issue, issue-active 68 -> 79 %, but 27 % more
    //  instructions because the straight-line form lets the compiler drop dead parts of every stage: 0.80 -> 0.87 ms)
    if constexpr (FP && !GEN) {
      step_backward_fp_lean<INTEG>(P, pl, x, rpm_cmd, lam, g_rpm);
    } else {
      float fd[3];
      disturbance(A.s0 + (uint32_t)t, fd);
      step_backward<MODEL, INTEG, OPT>(P, pl, x, FP ? rpm_cmd : acmd, fd, lam, FP ? g_rpm : g_acmd);
    }
    if (HAS_ATT) {
      if (att_phase == 0) {
        float g_prev[3];
        vjp_attitude_tick<OPT>(P, x + 3, x + 10, acmd, iR, g_rpm, g_iR, lam + 3, lam + 10, g_acmd, g_prev);
#pragma unroll
        for (int j = 0; j < 3; ++j) g_iR[j] = g_prev[j];
#pragma unroll
        for (int j = 0; j < 4; ++j) g_rpm[j] = 0.f;
      }
      att_phase = att_phase == 0 ? P.att_div - 1 : att_phase - 1;
    }
    if (POS) {
      if (pos_phase == 0) {           // the tick of this step produced att_cmd from (p, v, attitude, target, ip)
        float zB[3], gz[3] = { 0.f, 0.f, 0.f }, g_prev[3], sn[3], cs[3];
        if (FP) zB_fp(x + 3, zB); else zB_ab(x + 3, zB, sn, cs);
        vjp_position_tick(P, x, x + VEL, zB, cmd, ip, g_att, g_ip, lam, lam + VEL, gz, g_cmd, g_prev);
        if (FP) vjp_zB_fp(x + 3, gz, lam + 3); else vjp_zB_ab(sn, cs, gz, lam + 3);
#pragma unroll
        for (int j = 0; j < 3; ++j) g_ip[j] = g_prev[j];
#pragma unroll
        for (int j = 0; j < 4; ++j) g_att[j] = 0.f;
      }
      pos_phase = pos_phase == 0 ? P.pos_div - 1 : pos_phase - 1;
    }
    if (hold_phase == 0) {                                                     // the fetch step of command k_cmd
      if (FP && IFACE == IF_ROTOR) {
#pragma unroll
        for (int j = 0; j < 4; ++j) { g_cmd[j] = (cmd[j] > P.rpm_min && cmd[j] < P.rpm_max) ? g_rpm[j] : 0.f; g_rpm[j] = 0.f; }
      }
      if (FP && IFACE == IF_TORQUE) {                                          // the fetch ran the mixer on the command
        float g_tau[3];
        vjp_mixer<OPT>(P, cmd[3], cmd, g_rpm, &g_cmd[3], g_tau);
#pragma unroll
        for (int j = 0; j < 3; ++j) g_cmd[j] += g_tau[j];
#pragma unroll
        for (int j = 0; j < 4; ++j) g_rpm[j] = 0.f;
      }
      A.grad[(size_t)k_cmd * MN + i] = make_float4(g_cmd[0], g_cmd[1], g_cmd[2], g_cmd[3]);
#pragma unroll
      for (int j = 0; j < 4; ++j) g_cmd[j] = 0.f;
      hold_phase = A.cmd_hold - 1; --k_cmd;
    } else {
      --hold_phase;
    }
  }
}

struct Entry { int model, integ, iface; void (*fwd)(const GradArgs, const DevParams, int), (*bwd)(const GradArgs, const DevParams, int); };
#define CF_G(M_, I_, F_) { M_, I_, F_, grad_kernel<M_, I_, F_, 1>, grad_kernel<M_, I_, F_, 2> }
const Entry kTable[] = {
  CF_G(MODEL_FP, INTEG_EULER, IF_ATTITUDE), CF_G(MODEL_FP, INTEG_RK4, IF_ATTITUDE),
  CF_G(MODEL_FP, INTEG_EULER, IF_ROTOR),    CF_G(MODEL_FP, INTEG_RK4, IF_ROTOR),
  CF_G(MODEL_AB, INTEG_EULER, IF_ATTITUDE), CF_G(MODEL_AB, INTEG_RK4, IF_ATTITUDE),
  // the full onboard stack: position controller -> attitude controller -> mixer -> rotors
  CF_G(MODEL_FP, INTEG_EULER, IF_POSITION), CF_G(MODEL_FP, INTEG_RK4, IF_POSITION),
  CF_G(MODEL_AB, INTEG_EULER, IF_POSITION), CF_G(MODEL_AB, INTEG_RK4, IF_POSITION),
};
// the general kernels: fidelity extras, force disturbances (L280), torque interface (L330)
#define CF_GG(M_, I_, F_) { M_, I_, F_, grad_kernel<M_, I_, F_, 1, GOPT>, grad_kernel<M_, I_, F_, 2, GOPT> }
const Entry kTableGen[] = {
  CF_GG(MODEL_FP, INTEG_EULER, IF_ROTOR),    CF_GG(MODEL_FP, INTEG_RK4, IF_ROTOR),
  CF_GG(MODEL_FP, INTEG_EULER, IF_TORQUE),   CF_GG(MODEL_FP, INTEG_RK4, IF_TORQUE),
  CF_GG(MODEL_FP, INTEG_EULER, IF_ATTITUDE), CF_GG(MODEL_FP, INTEG_RK4, IF_ATTITUDE),
  CF_GG(MODEL_FP, INTEG_EULER, IF_POSITION), CF_GG(MODEL_FP, INTEG_RK4, IF_POSITION),
  CF_GG(MODEL_AB, INTEG_EULER, IF_ATTITUDE), CF_GG(MODEL_AB, INTEG_RK4, IF_ATTITUDE),
  CF_GG(MODEL_AB, INTEG_EULER, IF_POSITION), CF_GG(MODEL_AB, INTEG_RK4, IF_POSITION),
};
bool wants_general(const cf_sim *sim) {
  return (sim->opt & (OPT_DIST | OPT_EXTRAS)) != 0 || sim->p.iface == CF_IF_TORQUE;
}

int check(const cf_sim *sim, int n_cmds, int cmd_hold, int n_steps) {
  if (!sim) return fail(CF_E_ARG, "sim is NULL");
  if (n_steps < 1 || cmd_hold < 1 || n_cmds < 1) return fail(CF_E_ARG, "n_steps, cmd_hold, n_cmds >= 1");
  if ((long long)n_cmds * cmd_hold < n_steps) return fail(CF_E_SHAPE, "n_cmds * cmd_hold < n_steps");
  if (sim->p.cmd_source != CF_CMD_BUFFER || (sim->opt & OPT_NOISE) != 0)
    return fail(CF_E_UNSUPPORTED, "cf_grad differentiates the command-buffer rollout (the commands are its variables)");
  return CF_OK;
}

}  // namespace

static int hist_floats(int model, int iface, bool general) {
  if (general) return model == CF_MODEL_FIRST_PRINCIPLES ? Hist<MODEL_FP, IF_ATTITUDE, GOPT>::HD : Hist<MODEL_AB, IF_ATTITUDE, GOPT>::HD;
  if (model == CF_MODEL_FIRST_PRINCIPLES)
    return iface == CF_IF_POSITION ? Hist<MODEL_FP, IF_POSITION>::HD : iface == CF_IF_ATTITUDE ? Hist<MODEL_FP, IF_ATTITUDE>::HD
                                                                                               : Hist<MODEL_FP, IF_ROTOR>::HD;
  return iface == CF_IF_POSITION ? Hist<MODEL_AB, IF_POSITION>::HD : Hist<MODEL_AB, IF_ATTITUDE>::HD;
}

extern "C" size_t cf_grad_scratch_bytes(const cf_sim *sim, int n_steps) {
  if (!sim || n_steps < 1) return 0;
  return sizeof(float) * ((size_t)hist_floats(sim->model, sim->p.iface, wants_general(sim)) * (size_t)sim->MN * (size_t)n_steps + 4 + 4 * (size_t)sim->MN);
}

extern "C" int cf_grad(cf_sim *sim, const void *cmds_dev, int n_cmds, int cmd_hold, int n_steps, const float goal[3],
                       float *loss_dev, void *grad_dev, void *scratch_dev, size_t scratch_bytes) {
  int rc = check(sim, n_cmds, cmd_hold, n_steps);
  if (rc != CF_OK) return rc;
  if (!cmds_dev || !goal || !loss_dev || !grad_dev || !scratch_dev) return fail(CF_E_ARG, "NULL argument");
  if (!sim->have_state) return fail(CF_E_STATE, "cf_grad before cf_reset");
  if (((uintptr_t)cmds_dev & 15) || ((uintptr_t)grad_dev & 15) || ((uintptr_t)scratch_dev & 15))
    return fail(CF_E_BUFFER, "cmds, grad and scratch must be 16-byte aligned");
  if (scratch_bytes < cf_grad_scratch_bytes(sim, n_steps)) return fail(CF_E_BUFFER, "scratch too small");
  const Entry *e = nullptr;
  if (wants_general(sim)) {
    for (const Entry &c : kTableGen)
      if (c.model == sim->model && c.integ == sim->p.integrator && c.iface == sim->p.iface) e = &c;
  } else {
    for (const Entry &c : kTable)
      if (c.model == sim->model && c.integ == sim->p.integrator && c.iface == sim->p.iface) e = &c;
  }
  if (!e) return fail(CF_E_UNSUPPORTED, "cf_grad: the abstracted model has no rotor / torque interface");
  rc = cf_materialise(sim);      // a pending broadcast cf_set_state must be in the planes: the kernel reads them
  if (rc != CF_OK) return rc;
  GradArgs A;
  A.state = sim->state; A.ctrl = sim->ctrl; A.wparam = sim->wparam;
  A.cmds = (const float4 *)cmds_dev; A.grad = (float4 *)grad_dev; A.loss = loss_dev; A.hist = (float4 *)scratch_dev;
  A.MN = sim->MN; A.M = sim->M; A.N = sim->N; A.n_steps = n_steps; A.cmd_hold = cmd_hold; A.n_cmds = n_cmds;
  A.s0 = (uint32_t)sim->s_host;
  for (int j = 0; j < 3; ++j) A.goal[j] = goal[j];
  A.world_offset = sim->p.world_offset;
  const uint32_t lo = (uint32_t)sim->seed, hi = (uint32_t)(sim->seed >> 32);
  for (int r = 0; r < 10; ++r) { A.rk[2 * r] = lo + (uint32_t)r * 0x9E3779B9u; A.rk[2 * r + 1] = hi + (uint32_t)r * 0xBB67AE85u; }
  const int block = 128;
  const unsigned grid = (unsigned)((sim->MN + block - 1) / block);
  e->fwd<<<grid, block, 0, sim->stream>>>(A, sim->dp, (sim->opt & OPT_RANDP) ? 1 : 0);
  e->bwd<<<grid, block, 0, sim->stream>>>(A, sim->dp, (sim->opt & OPT_RANDP) ? 1 : 0);
  CF_CUDA(cudaGetLastError());
  // commands beyond the last used one get a zero gradient
  int used = (n_steps + cmd_hold - 1) / cmd_hold;
  if (used < n_cmds)
    CF_CUDA(cudaMemsetAsync((float4 *)grad_dev + (size_t)used * sim->MN, 0, sizeof(float4) * (size_t)(n_cmds - used) * sim->MN, sim->stream));
  return CF_OK;
}

// The same call driven from HOST buffers (the end-to-end path): commands host->device into staging_dev, the kernel, loss
// and gradient device->host, stream synchronised.  staging_dev: cf_grad_staging_bytes() bytes, 256-byte aligned.
static size_t align256g(size_t n) { return (n + 255) & ~(size_t)255; }
extern "C" size_t cf_grad_staging_bytes(const cf_sim *sim, int n_cmds) {
  if (!sim || n_cmds < 1) return 0;
  const size_t cb = align256g(sizeof(float) * 4 * (size_t)sim->MN * (size_t)n_cmds);
  return 2 * cb + align256g(sizeof(float) * (size_t)sim->MN);
}
extern "C" int cf_grad_host(cf_sim *sim, const void *cmds_host, int n_cmds, int cmd_hold, int n_steps, const float goal[3],
                            float *loss_host, void *grad_host, void *staging_dev, size_t staging_bytes, void *scratch_dev,
                            size_t scratch_bytes) {
  if (!sim || !cmds_host || !loss_host || !grad_host || !staging_dev) return fail(CF_E_ARG, "NULL argument");
  if (n_cmds < 1) return fail(CF_E_ARG, "n_cmds >= 1");
  if (((uintptr_t)staging_dev & 255) != 0) return fail(CF_E_BUFFER, "staging must be 256-byte aligned");
  if (staging_bytes < cf_grad_staging_bytes(sim, n_cmds)) return fail(CF_E_BUFFER, "staging too small");
  const size_t raw = sizeof(float) * 4 * (size_t)sim->MN * (size_t)n_cmds, cb = align256g(raw);
  char *base = (char *)staging_dev;
  void *cmds_dev = base, *grad_dev = base + cb;
  float *loss_dev = (float *)(base + 2 * cb);
  CF_CUDA(cudaMemcpyAsync(cmds_dev, cmds_host, raw, cudaMemcpyHostToDevice, sim->stream));
  int rc = cf_grad(sim, cmds_dev, n_cmds, cmd_hold, n_steps, goal, loss_dev, grad_dev, scratch_dev, scratch_bytes);
  if (rc != CF_OK) return rc;
  CF_CUDA(cudaMemcpyAsync(grad_host, grad_dev, raw, cudaMemcpyDeviceToHost, sim->stream));
  CF_CUDA(cudaMemcpyAsync(loss_host, loss_dev, sizeof(float) * (size_t)sim->MN, cudaMemcpyDeviceToHost, sim->stream));
  CF_CUDA(cudaStreamSynchronize(sim->stream));
  return CF_OK;
}
