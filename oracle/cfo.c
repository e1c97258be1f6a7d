/* cfo.c -- float64 CPU ORACLE (test infrastructure; see cfo.h for the contract and layouts).
 *
 * Written from PAPER.md: rigid body Eqs. (1)-(4) (L300-L309), rotor thrust / torque polynomials and
 * mixing matrix (L311-L315), gyroscopic / reaction torque Eq. (5) (L313), body drag (L317), rotor
 * dynamics Eq. (6) (L321), abstracted model Eqs. (7)-(10) (L344-L354), control interfaces (L330),
 * geometric position controller (L356).  Where the paper is silent the numbered readings of
 * DESIGN.md apply (R1..R24, the same list as SURVEY.md 8(c) G1..G24); they are quoted at each use.
 *
 * No blocking, fusion, reordering or fast-math: one drone at a time, one step at a time, in the
 * order of DESIGN.md "Per-step order" (C8).  OpenMP only over drones (they are independent).
 */
#include "cfo.h"
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define PI 3.14159265358979323846

struct cfo_sim {
  int64_t M, N, MN;
  int model, D, P;
  cfo_params p;
  double *x;      /* [D][MN]  */
  double *ctrl;   /* [14][MN] */
  double *wp;     /* [P][M]   */
  double *mind2;  /* [8][MN]  */
  double *eps;    /* [4][MN] AR(1) command-noise state, NaN = none drawn since the last re-arm (R25) */
  double *cost;   /* [MN] running rollout cost (R27) */
  uint32_t s, att_ticks, pos_ticks, n_rec_total;
  uint32_t rec_table[CFO_REC_TABLE_CAP];
  uint64_t seed;
  int have_state;
};

static int g_threads = 0;
int cfo_num_threads(void) {
#ifdef _OPENMP
  return g_threads > 0 ? g_threads : omp_get_max_threads();
#else
  return 1;
#endif
}
void cfo_set_num_threads(int n) { g_threads = n; }

int cfo_state_dim(int model) { return model == CFO_MODEL_FIRST_PRINCIPLES ? 17 : 13; }
int cfo_world_param_dim(int model) { return model == CFO_MODEL_FIRST_PRINCIPLES ? 14 : 11; }

/* ------------------------------------------------------------------------------------------ */
/* C0 constants: BASELINE.json configs[0] and configs[2]; limits and gains are readings R7,R12,R16 */
void cfo_default_params(cfo_params *p, int model) {
  memset(p, 0, sizeof(*p));
  p->integrator = CFO_EULER;
  p->iface = CFO_IF_ATTITUDE;
  p->cmd_source = CFO_CMD_BUFFER;
  p->ab_thrust_dyn = 1;
  p->f_phys = model == CFO_MODEL_FIRST_PRINCIPLES ? 1000.0 : 500.0;
  p->f_att = 500.0;
  p->f_pos = 100.0;
  p->mass = 0.027;
  p->J[0] = 1.395e-5; p->J[1] = 1.395e-5; p->J[2] = 2.173e-5;
  p->arm = 0.046;
  p->kf[2] = 3.16e-10;
  p->km[2] = 7.94e-12;
  p->g = 9.81;
  p->cv_up = 1.0 / 0.03; p->cv_dn = 1.0 / 0.03;
  for (int j = 0; j < 3; ++j) { p->ab_a[j] = -130.0; p->ab_b[j] = -16.0; p->ab_c[j] = 130.0; }
  p->ab_ctau = 1.0 / 0.03; p->ab_cf = 1.0;
  p->rpm_min = 0.0; p->rpm_max = 21700.0; p->thrust_min = 0.0; p->thrust_max = 0.55; p->tilt_max = 0.5;
  for (int j = 0; j < 3; ++j) { p->kR[j] = 130.0; p->kW[j] = 16.0; }
  p->kI[0] = 20.0; p->kI[1] = 20.0; p->kI[2] = 0.0; p->iR_max = 0.2;
  p->kp[0] = 8; p->kp[1] = 8; p->kp[2] = 12;
  p->kd[0] = 5; p->kd[1] = 5; p->kd[2] = 7;
  p->ki[0] = 1; p->ki[1] = 1; p->ki[2] = 6;
  p->ip_max[0] = 0.25; p->ip_max[1] = 0.25; p->ip_max[2] = 0.4;
  for (int j = 0; j < 12; ++j) { p->rnd_lo[j] = 1.0; p->rnd_hi[j] = 1.0; }
  p->p0_lo[2] = 1.0; p->p0_hi[2] = 1.0;
  p->grid_dims[0] = p->grid_dims[1] = p->grid_dims[2] = 1;
  p->cmd_lo[0] = -0.5; p->cmd_lo[1] = -0.5; p->cmd_lo[2] = -PI; p->cmd_lo[3] = 0.05;
  p->cmd_hi[0] = 0.5;  p->cmd_hi[1] = 0.5;  p->cmd_hi[2] = PI;  p->cmd_hi[3] = 0.55;
  p->n_ctrl = 1;
}

static double clipd(double v, double lo, double hi) { return v < lo ? lo : (v > hi ? hi : v); }

/* ------------------------------------------------------------------------------------------ */
/* C9: Philox4x32-10 (Salmon et al. 2011).  key = (seed lo, seed hi). */
void cfo_philox(uint64_t seed, const uint32_t ctr[4], uint32_t out[4]) {
  uint32_t k0 = (uint32_t)(seed & 0xFFFFFFFFu), k1 = (uint32_t)(seed >> 32);
  uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
  for (int r = 0; r < 10; ++r) {
    if (r > 0) { k0 += 0x9E3779B9u; k1 += 0xBB67AE85u; }
    uint64_t p0 = (uint64_t)0xD2511F53u * c0;
    uint64_t p1 = (uint64_t)0xCD9E8D57u * c2;
    uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
    uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
    uint32_t n0 = hi1 ^ c1 ^ k0, n1 = lo1, n2 = hi0 ^ c3 ^ k1, n3 = lo0;
    c0 = n0; c1 = n1; c2 = n2; c3 = n3;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}
/* R18: 23-bit midpoint uniform in (0,1), exact in float32 and float64 */
double cfo_uniform(uint32_t x) { return ((double)(x >> 9) + 0.5) * (1.0 / 8388608.0); }
/* Box-Muller, C9 */
void cfo_normal_pair(uint32_t xa, uint32_t xb, double *z0, double *z1) {
  double ua = cfo_uniform(xa), ub = cfo_uniform(xb);
  double r = sqrt(-2.0 * log(ua));
  *z0 = r * cos(2.0 * PI * ub);
  *z1 = r * sin(2.0 * PI * ub);
}
enum { STREAM_INIT = 0, STREAM_PARAM = 1, STREAM_DIST = 2, STREAM_NOISE = 3 };
static void philox_at(uint64_t seed, int64_t w, int64_t n, uint32_t index, uint32_t stream, uint32_t out[4]) {
  uint32_t c[4] = { (uint32_t)w, (uint32_t)n, index, stream };
  cfo_philox(seed, c, out);
}

/* ------------------------------------------------------------------------------------------ */
/* rotations */
static void quat_to_R(const double q[4], double R[3][3]) {   /* scalar-last (x,y,z,w) */
  double x = q[0], y = q[1], z = q[2], w = q[3];
  R[0][0] = 1 - 2 * (y * y + z * z); R[0][1] = 2 * (x * y - w * z);     R[0][2] = 2 * (x * z + w * y);
  R[1][0] = 2 * (x * y + w * z);     R[1][1] = 1 - 2 * (x * x + z * z); R[1][2] = 2 * (y * z - w * x);
  R[2][0] = 2 * (x * z - w * y);     R[2][1] = 2 * (y * z + w * x);     R[2][2] = 1 - 2 * (x * x + y * y);
}
/* R13: R = Rz(yaw) Ry(pitch) Rx(roll) */
static void euler_to_R(double roll, double pitch, double yaw, double R[3][3]) {
  double cr = cos(roll), sr = sin(roll), cp = cos(pitch), sp = sin(pitch), cy = cos(yaw), sy = sin(yaw);
  R[0][0] = cy * cp; R[0][1] = cy * sp * sr - sy * cr; R[0][2] = cy * sp * cr + sy * sr;
  R[1][0] = sy * cp; R[1][1] = sy * sp * sr + cy * cr; R[1][2] = sy * sp * cr - cy * sr;
  R[2][0] = -sp;     R[2][1] = cp * sr;                R[2][2] = cp * cr;
}
static void cross3(const double a[3], const double b[3], double c[3]) {
  c[0] = a[1] * b[2] - a[2] * b[1]; c[1] = a[2] * b[0] - a[0] * b[2]; c[2] = a[0] * b[1] - a[1] * b[0];
}
static double norm3(const double a[3]) { return sqrt(a[0] * a[0] + a[1] * a[1] + a[2] * a[2]); }

/* ------------------------------------------------------------------------------------------ */
/* C1: X-configuration mixing matrix (R5, R6).  Rotor k at lever*(+1,-1), (-1,-1), (-1,+1), (+1,+1);
 * spin d = (+,-,+,-) about body +z (sign pattern of Eq. (5)). */
static const double SX[4] = { -1, -1, +1, +1 };
static const double SY[4] = { -1, +1, +1, -1 };
static const double SZ[4] = { -1, +1, -1, +1 };   /* = -d */
static const double DSPIN[4] = { +1, -1, +1, -1 };

static double poly2(const double c[3], double x) { return c[0] + c[1] * x + c[2] * x * x; }

typedef struct {   /* plant parameters of one world */
  double m, J[3], kf[3], km[3], cv_up, cv_dn, cd_up, cd_dn;
  double a[3], b[3], c[3], ctau;
} plant_t;

static void mix_forward(const double kf[3], const double km[3], double lever, const double rpm[4],
                        double *F, double tau[3]) {
  double f[4], mk[4];
  for (int k = 0; k < 4; ++k) { f[k] = poly2(kf, rpm[k]); mk[k] = poly2(km, rpm[k]); }
  *F = f[0] + f[1] + f[2] + f[3];
  tau[0] = lever * (SX[0] * f[0] + SX[1] * f[1] + SX[2] * f[2] + SX[3] * f[3]);
  tau[1] = lever * (SY[0] * f[0] + SY[1] * f[1] + SY[2] * f[2] + SY[3] * f[3]);
  tau[2] = SZ[0] * mk[0] + SZ[1] * mk[1] + SZ[2] * mk[2] + SZ[3] * mk[3];
}
void cfo_mix(const cfo_params *p, const double rpm[4], double *F, double tau[3]) {
  mix_forward(p->kf, p->km, p->arm / sqrt(2.0), rpm, F, tau);
}

/* C2: first-principles derivative, Eqs. (1)-(6) */
static void deriv_fp(const cfo_params *p, const plant_t *pl, const double x[17], const double rpm_cmd[4],
                     const double fdist[3], double dx[17]) {
  const double *q = x + 3, *v = x + 7, *w = x + 10, *Om = x + 13;
  double dOm[4];
  /* 1. rotor dynamics Eq. (6): branch on the sign of the speed error, re-evaluated at every stage */
  for (int k = 0; k < 4; ++k) {
    double e = rpm_cmd[k] - Om[k];
    double cv = e >= 0 ? pl->cv_up : pl->cv_dn, cd = e >= 0 ? pl->cd_up : pl->cd_dn;
    dOm[k] = cv * e + cd * (rpm_cmd[k] * rpm_cmd[k] - Om[k] * Om[k]);
  }
  /* 2. thrust / drag-torque polynomials and mixing matrix */
  double F, tau[3];
  mix_forward(pl->kf, pl->km, p->arm / sqrt(2.0), Om, &F, tau);
  /* 3. gyroscopic + reaction torque Eq. (5), reading R2: Jp(-wy S, +wx S, -dS), rpm -> rad/s (R3) */
  if (p->Jp != 0.0) {
    double S = 0, dS = 0;
    for (int k = 0; k < 4; ++k) { S += DSPIN[k] * Om[k]; dS += DSPIN[k] * dOm[k]; }
    S *= 2.0 * PI / 60.0; dS *= 2.0 * PI / 60.0;
    tau[0] += p->Jp * (-w[1] * S);
    tau[1] += p->Jp * (+w[0] * S);
    tau[2] += p->Jp * (-dS);
  }
  /* 4. Eq. (3): m dv = R e_z F + f_dist + R (Ca .* (R^T v)) - m g e_z */
  double R[3][3];
  quat_to_R(q, R);
  double fw[3] = { R[0][2] * F + fdist[0], R[1][2] * F + fdist[1], R[2][2] * F + fdist[2] };
  if (p->Ca[0] != 0.0 || p->Ca[1] != 0.0 || p->Ca[2] != 0.0) {
    double vb[3], fb[3];
    for (int j = 0; j < 3; ++j) vb[j] = R[0][j] * v[0] + R[1][j] * v[1] + R[2][j] * v[2];
    for (int j = 0; j < 3; ++j) fb[j] = p->Ca[j] * vb[j];
    for (int i = 0; i < 3; ++i) fw[i] += R[i][0] * fb[0] + R[i][1] * fb[1] + R[i][2] * fb[2];
  }
  dx[7] = fw[0] / pl->m; dx[8] = fw[1] / pl->m; dx[9] = fw[2] / pl->m - p->g;
  /* 5. Eq. (4): J dw = tau - w x (J w), diagonal J */
  double Jw[3] = { pl->J[0] * w[0], pl->J[1] * w[1], pl->J[2] * w[2] }, wxJw[3];
  cross3(w, Jw, wxJw);
  for (int j = 0; j < 3; ++j) dx[10 + j] = (tau[j] - wxJw[j]) / pl->J[j];
  /* 6. Eq. (2), reading R1: dq = 1/2 q (x) (w, 0), Hamilton product, scalar-last */
  double qv[3] = { q[0], q[1], q[2] }, qvxw[3];
  cross3(qv, w, qvxw);
  for (int j = 0; j < 3; ++j) dx[3 + j] = 0.5 * (q[3] * w[j] + qvxw[j]);
  dx[6] = -0.5 * (qv[0] * w[0] + qv[1] * w[1] + qv[2] * w[2]);
  /* 7. Eq. (1) */
  dx[0] = v[0]; dx[1] = v[1]; dx[2] = v[2];
  for (int k = 0; k < 4; ++k) dx[13 + k] = dOm[k];
}

/* C3: abstracted derivative, Eqs. (7)-(10); u = (roll_c, pitch_c, yaw_c, f_c) */
static void deriv_ab(const cfo_params *p, const plant_t *pl, const double x[13], const double u[4],
                     const double fdist[3], double dx[13]) {
  const double *Psi = x + 3, *v = x + 6, *dPsi = x + 9;
  double R[3][3];
  euler_to_R(Psi[0], Psi[1], Psi[2], R);
  double fS = p->ab_thrust_dyn ? x[12] : u[3];          /* simplified variant */
  double T = p->ab_cf * fS;
  double fw[3] = { R[0][2] * T + fdist[0], R[1][2] * T + fdist[1], R[2][2] * T + fdist[2] };
  if (p->Ca[0] != 0.0 || p->Ca[1] != 0.0 || p->Ca[2] != 0.0) {
    double vb[3], fb[3];
    for (int j = 0; j < 3; ++j) vb[j] = R[0][j] * v[0] + R[1][j] * v[1] + R[2][j] * v[2];
    for (int j = 0; j < 3; ++j) fb[j] = p->Ca[j] * vb[j];
    for (int i = 0; i < 3; ++i) fw[i] += R[i][0] * fb[0] + R[i][1] * fb[1] + R[i][2] * fb[2];
  }
  dx[0] = v[0]; dx[1] = v[1]; dx[2] = v[2];                                   /* Eq. (7) */
  dx[6] = fw[0] / pl->m; dx[7] = fw[1] / pl->m; dx[8] = fw[2] / pl->m - p->g; /* Eq. (8) */
  for (int j = 0; j < 3; ++j) {
    dx[3 + j] = dPsi[j];                                                      /* Euler-angle rates */
    dx[9 + j] = pl->a[j] * Psi[j] + pl->b[j] * dPsi[j] + pl->c[j] * u[j];     /* Eq. (10) */
  }
  dx[12] = p->ab_thrust_dyn ? pl->ctau * (u[3] - x[12]) : 0.0;                /* Eq. (9) */
}

static void deriv(const cfo_sim *S, const plant_t *pl, const double *x, const double *u,
                  const double fdist[3], double *dx) {
  if (S->model == CFO_MODEL_FIRST_PRINCIPLES) deriv_fp(&S->p, pl, x, u, fdist, dx);
  else deriv_ab(&S->p, pl, x, u, fdist, dx);
}

/* C4: explicit Euler / classical RK4 with zero-order-held inputs; stage quaternions not renormalised;
 * q <- q/|q| once after the full step (R8-R10). */
static void integrate(const cfo_sim *S, const plant_t *pl, double *x, const double *u, const double fdist[3]) {
  const int D = S->D;
  const double h = 1.0 / S->p.f_phys;
  double k1[17], k2[17], k3[17], k4[17], xs[17];
  if (S->p.integrator == CFO_EULER) {
    deriv(S, pl, x, u, fdist, k1);
    for (int j = 0; j < D; ++j) x[j] = x[j] + h * k1[j];
  } else {
    deriv(S, pl, x, u, fdist, k1);
    for (int j = 0; j < D; ++j) xs[j] = x[j] + 0.5 * h * k1[j];
    deriv(S, pl, xs, u, fdist, k2);
    for (int j = 0; j < D; ++j) xs[j] = x[j] + 0.5 * h * k2[j];
    deriv(S, pl, xs, u, fdist, k3);
    for (int j = 0; j < D; ++j) xs[j] = x[j] + h * k3[j];
    deriv(S, pl, xs, u, fdist, k4);
    for (int j = 0; j < D; ++j) x[j] = x[j] + h / 6.0 * (k1[j] + 2.0 * k2[j] + 2.0 * k3[j] + k4[j]);
  }
  if (S->model == CFO_MODEL_FIRST_PRINCIPLES) {
    double *q = x + 3, nq = sqrt(q[0] * q[0] + q[1] * q[1] + q[2] * q[2] + q[3] * q[3]);
    for (int j = 0; j < 4; ++j) q[j] /= nq;
  } else if (!S->p.ab_thrust_dyn) {
    x[12] = u[3];   /* f_Sigma == f_cmd in the simplified variant */
  }
}

/* inverse of the nominal thrust polynomial f = kf0 + kf1 W + kf2 W^2 (positive root) */
static double thrust_to_rpm(const double kf[3], double f) {
  if (kf[0] == 0.0 && kf[1] == 0.0) return sqrt(f / kf[2]);
  double disc = kf[1] * kf[1] - 4.0 * kf[2] * (kf[0] - f);
  if (disc < 0) disc = 0;
  return (-kf[1] + sqrt(disc)) / (2.0 * kf[2]);
}

/* C6 mixer (R5, R12): (F_c, tau_des) -> rotor thrusts -> clip -> rpm -> clip.  Nominal parameters (R11). */
static void mixer(const cfo_params *p, double Fc, const double tau[3], double rpm_cmd[4]) {
  double lever = p->arm / sqrt(2.0), kappa = p->km[2] / p->kf[2];
  double fmax = poly2(p->kf, p->rpm_max);
  for (int k = 0; k < 4; ++k) {
    double f = Fc / 4.0 + (SX[k] * tau[0] + SY[k] * tau[1]) / (4.0 * lever) + SZ[k] * tau[2] / (4.0 * kappa);
    f = clipd(f, 0.0, fmax);
    rpm_cmd[k] = clipd(thrust_to_rpm(p->kf, f), p->rpm_min, p->rpm_max);
  }
}

/* C5 attitude controller tick (R7).  cmd = (roll, pitch, yaw, thrust). */
void cfo_attitude_tick(const cfo_params *p, const double q[4], const double w[3], const double cmd[4],
                       double iR[3], double eR_out[3], double tau_out[3], double rpm_cmd[4]) {
  double hatt = (p->f_phys / p->f_att) * (1.0 / p->f_phys);   /* att_div * h */
  double Rd[3][3], R[3][3], Mx[3][3];
  euler_to_R(cmd[0], cmd[1], cmd[2], Rd);
  quat_to_R(q, R);
  for (int i = 0; i < 3; ++i)
    for (int j = 0; j < 3; ++j) Mx[i][j] = Rd[0][i] * R[0][j] + Rd[1][i] * R[1][j] + Rd[2][i] * R[2][j];  /* Rd^T R */
  double eR[3] = { 0.5 * (Mx[2][1] - Mx[1][2]), 0.5 * (Mx[0][2] - Mx[2][0]), 0.5 * (Mx[1][0] - Mx[0][1]) };
  double tau[3];
  for (int j = 0; j < 3; ++j) {
    iR[j] = clipd(iR[j] + eR[j] * hatt, -p->iR_max, p->iR_max);          /* updated before use */
    tau[j] = p->J[j] * (-p->kR[j] * eR[j] - p->kW[j] * w[j] - p->kI[j] * iR[j]);
  }
  mixer(p, cmd[3], tau, rpm_cmd);
  if (eR_out) for (int j = 0; j < 3; ++j) eR_out[j] = eR[j];
  if (tau_out) for (int j = 0; j < 3; ++j) tau_out[j] = tau[j];
}

/* C7 geometric position controller tick (R16).  target = (x, y, z, yaw). */
void cfo_position_tick(const cfo_params *p, const double pos[3], const double vel[3], const double zB[3],
                       const double target[4], double ip[3], double att_cmd[4]) {
  double hpos = (p->f_phys / p->f_pos) * (1.0 / p->f_phys);
  double t[3];
  for (int j = 0; j < 3; ++j) {
    double ep = target[j] - pos[j], ev = -vel[j];
    ip[j] = clipd(ip[j] + ep * hpos, -p->ip_max[j], p->ip_max[j]);
    double ad = p->kp[j] * ep + p->kd[j] * ev + p->ki[j] * ip[j] + (j == 2 ? p->g : 0.0);
    t[j] = p->mass * ad;
  }
  double Fc = clipd(t[0] * zB[0] + t[1] * zB[1] + t[2] * zB[2], p->thrust_min, p->thrust_max);
  double nt = fmax(norm3(t), 1e-6);
  double zd[3] = { t[0] / nt, t[1] / nt, t[2] / nt };
  double xc[3] = { cos(target[3]), sin(target[3]), 0.0 }, yd[3], xd[3];
  cross3(zd, xc, yd);
  double ny = fmax(norm3(yd), 1e-6);
  for (int j = 0; j < 3; ++j) yd[j] /= ny;
  cross3(yd, zd, xd);
  att_cmd[0] = clipd(atan2(yd[2], zd[2]), -p->tilt_max, p->tilt_max);
  att_cmd[1] = clipd(asin(clipd(-xd[2], -1.0, 1.0)), -p->tilt_max, p->tilt_max);
  att_cmd[2] = atan2(xd[1], xd[0]);
  att_cmd[3] = Fc;
}

/* ------------------------------------------------------------------------------------------ */
static double hover_rpm(const cfo_params *p) { return thrust_to_rpm(p->kf, p->mass * p->g / 4.0); }

static void load_plant(const cfo_sim *S, int64_t w, plant_t *pl) {
  const double *wp = S->wp; const int64_t M = S->M;
  memset(pl, 0, sizeof(*pl));
  if (S->model == CFO_MODEL_FIRST_PRINCIPLES) {
    pl->m = wp[0 * M + w];
    for (int j = 0; j < 3; ++j) { pl->J[j] = wp[(1 + j) * M + w]; pl->kf[j] = wp[(4 + j) * M + w]; pl->km[j] = wp[(7 + j) * M + w]; }
    pl->cv_up = wp[10 * M + w]; pl->cv_dn = wp[11 * M + w]; pl->cd_up = wp[12 * M + w]; pl->cd_dn = wp[13 * M + w];
  } else {
    pl->m = wp[0 * M + w];
    for (int j = 0; j < 3; ++j) { pl->a[j] = wp[(1 + j) * M + w]; pl->b[j] = wp[(4 + j) * M + w]; pl->c[j] = wp[(7 + j) * M + w]; }
    pl->ctau = wp[10 * M + w];
  }
}

int cfo_create(cfo_sim **out, int64_t M, int64_t N, int model, const cfo_params *p) {
  if (!out || !p || M < 1 || N < 1 || (model != 0 && model != 1)) return -1;
  if (M * N >= ((int64_t)1 << 31)) return -2;
  double ad = p->f_phys / p->f_att, pd = p->f_phys / p->f_pos;
  if (p->f_phys <= 0 || ad < 1 || pd < 1 || ad != floor(ad) || pd != floor(pd)) return -1;
  if (model == CFO_MODEL_ABSTRACTED && p->iface != CFO_IF_ATTITUDE && p->iface != CFO_IF_POSITION) return -6;
  if (p->n_obstacles < 0 || p->n_obstacles > 8) return -1;
  if (!(p->noise_beta >= 0.0 && p->noise_beta < 1.0) || p->n_ctrl < 1 || p->worlds_per_ctrl < 0) return -1;
  cfo_sim *S = (cfo_sim *)calloc(1, sizeof(cfo_sim));
  S->M = M; S->N = N; S->MN = M * N; S->model = model; S->p = *p;
  S->D = cfo_state_dim(model); S->P = cfo_world_param_dim(model);
  S->x = (double *)calloc((size_t)S->D * S->MN, sizeof(double));
  S->ctrl = (double *)calloc((size_t)14 * S->MN, sizeof(double));
  S->wp = (double *)calloc((size_t)S->P * M, sizeof(double));
  S->mind2 = (double *)calloc((size_t)8 * S->MN, sizeof(double));
  S->eps = (double *)calloc((size_t)4 * S->MN, sizeof(double));
  S->cost = (double *)calloc((size_t)S->MN, sizeof(double));
  *out = S;
  return 0;
}
void cfo_destroy(cfo_sim *S) {
  if (!S) return;
  free(S->x); free(S->ctrl); free(S->wp); free(S->mind2); free(S->eps); free(S->cost); free(S);
}

static void rearm_drone(cfo_sim *S, int64_t i) {
  /* integrals 0, held commands = hover of the nominal model, min distance +inf (R20) */
  const cfo_params *p = &S->p;
  double wh = S->model == CFO_MODEL_FIRST_PRINCIPLES ? hover_rpm(p) : 0.0;
  for (int c = 0; c < 9; ++c) S->ctrl[c * S->MN + i] = 0.0;
  S->ctrl[9 * S->MN + i] = p->mass * p->g;
  for (int k = 0; k < 4; ++k) S->ctrl[(10 + k) * S->MN + i] = wh;
  for (int j = 0; j < 8; ++j) S->mind2[j * S->MN + i] = INFINITY;
  for (int j = 0; j < 4; ++j) S->eps[j * S->MN + i] = NAN;   /* R25: the next command starts a fresh noise chain */
  S->cost[i] = 0.0;                                          /* R27 */
}
static void rearm_controllers(cfo_sim *S) {
  for (int64_t i = 0; i < S->MN; ++i) rearm_drone(S, i);
}

static void reset_world_state(cfo_sim *S, uint64_t seed, int64_t w);

/* C9 reset: PARAM stream (world params) + INIT stream (initial state) */
int cfo_reset(cfo_sim *S, uint64_t seed) {
  if (!S) return -1;
  const cfo_params *p = &S->p;
  const int64_t M = S->M, N = S->N, MN = S->MN;
  S->seed = seed;
  for (int64_t w = 0; w < M; ++w) {
    int64_t wg = w + p->world_offset;
    double fac[12];
    for (int b = 0; b < 3; ++b) {
      uint32_t r[4];
      philox_at(seed, wg, 0, (uint32_t)b, STREAM_PARAM, r);
      for (int k = 0; k < 4; ++k) {
        int slot = 4 * b + k;
        fac[slot] = p->rnd_lo[slot] + (p->rnd_hi[slot] - p->rnd_lo[slot]) * cfo_uniform(r[k]);
      }
    }
    double *wp = S->wp;
    if (S->model == CFO_MODEL_FIRST_PRINCIPLES) {     /* R17: slots (m,Jx,Jy,Jz | kf,km,tau_m,-) */
      wp[0 * M + w] = p->mass * fac[0];
      for (int j = 0; j < 3; ++j) wp[(1 + j) * M + w] = p->J[j] * fac[1 + j];
      for (int j = 0; j < 3; ++j) wp[(4 + j) * M + w] = p->kf[j] * fac[4];
      for (int j = 0; j < 3; ++j) wp[(7 + j) * M + w] = p->km[j] * fac[5];
      wp[10 * M + w] = p->cv_up / fac[6]; wp[11 * M + w] = p->cv_dn / fac[6];
      wp[12 * M + w] = p->cd_up / fac[6]; wp[13 * M + w] = p->cd_dn / fac[6];
    } else {                                           /* slots (m,a[3] | b[3],- | c[3],c_tau) */
      wp[0 * M + w] = p->mass * fac[0];
      for (int j = 0; j < 3; ++j) wp[(1 + j) * M + w] = p->ab_a[j] * fac[1 + j];
      for (int j = 0; j < 3; ++j) wp[(4 + j) * M + w] = p->ab_b[j] * fac[4 + j];
      for (int j = 0; j < 3; ++j) wp[(7 + j) * M + w] = p->ab_c[j] * fac[8 + j];
      wp[10 * M + w] = p->ab_ctau * fac[11];
    }
  }
  for (int64_t w = 0; w < M; ++w) reset_world_state(S, seed, w);
  rearm_controllers(S);
  S->s = 0; S->att_ticks = 0; S->pos_ticks = 0; S->n_rec_total = 0;
  memset(S->rec_table, 0, sizeof(S->rec_table));
  S->have_state = 1;
  return 0;
}

/* Continuous environment resets: the worlds with mask[w] != 0 start a new episode -- initial state
 * re-drawn from the INIT stream of `episode_seed`, controllers re-armed -- while the other worlds, the per-world
 * parameters, the step counter and the seed of the disturbance / noise streams stay as they are. */
int cfo_reset_masked(cfo_sim *S, const uint8_t *mask, uint64_t episode_seed) {
  if (!S || !mask) return -1;
  if (!S->have_state) return -3;
  for (int64_t w = 0; w < S->M; ++w) {
    if (!mask[w]) continue;
    reset_world_state(S, episode_seed, w);
    for (int64_t n = 0; n < S->N; ++n) rearm_drone(S, w * S->N + n);
  }
  return 0;
}

/* INIT stream -> initial state of the drones of world w (C9) */
static void reset_world_state(cfo_sim *S, uint64_t seed, int64_t w) {
  const cfo_params *p = &S->p;
  const int64_t N = S->N, MN = S->MN;
  {
    int64_t wg = w + p->world_offset;
    for (int64_t n = 0; n < N; ++n) {
      int64_t i = w * N + n;
      double pos[3], q[4] = { 0, 0, 0, 1 };
      uint32_t r[4];
      if (p->init_mode == 0) {
        for (int j = 0; j < 3; ++j) pos[j] = p->p0_lo[j];
      } else if (p->init_mode == 1) {
        philox_at(seed, wg, n, 0, STREAM_INIT, r);
        for (int j = 0; j < 3; ++j) pos[j] = p->p0_lo[j] + (p->p0_hi[j] - p->p0_lo[j]) * cfo_uniform(r[j]);
        philox_at(seed, wg, n, 1, STREAM_INIT, r);                       /* R19 */
        double zeta = 2.0 * cfo_uniform(r[0]) - 1.0, alpha = 2.0 * PI * cfo_uniform(r[1]);
        double theta = p->tilt0_max * cfo_uniform(r[2]);
        double sxy = sqrt(1.0 - zeta * zeta);
        double ax[3] = { sxy * cos(alpha), sxy * sin(alpha), zeta };
        double sh = sin(0.5 * theta);
        q[0] = ax[0] * sh; q[1] = ax[1] * sh; q[2] = ax[2] * sh; q[3] = cos(0.5 * theta);
      } else {
        philox_at(seed, wg, n, 0, STREAM_INIT, r);
        int64_t gx = p->grid_dims[0], gy = p->grid_dims[1];
        int64_t cell[3] = { n % gx, (n / gx) % gy, n / (gx * gy) };
        for (int j = 0; j < 3; ++j)
          pos[j] = p->grid_origin[j] + p->grid_spacing * (double)cell[j] + p->grid_jitter * (2.0 * cfo_uniform(r[j]) - 1.0);
      }
      double *x = S->x;
      for (int j = 0; j < S->D; ++j) x[j * MN + i] = 0.0;
      for (int j = 0; j < 3; ++j) x[j * MN + i] = pos[j];
      if (S->model == CFO_MODEL_FIRST_PRINCIPLES) {
        for (int j = 0; j < 4; ++j) x[(3 + j) * MN + i] = q[j];
        double wh = hover_rpm(p);
        for (int k = 0; k < 4; ++k) x[(13 + k) * MN + i] = wh;
      } else {
        double R[3][3];
        quat_to_R(q, R);
        x[3 * MN + i] = atan2(R[2][1], R[2][2]);
        x[4 * MN + i] = -asin(clipd(R[2][0], -1.0, 1.0));
        x[5 * MN + i] = atan2(R[1][0], R[0][0]);
        x[12 * MN + i] = p->mass * p->g;
      }
    }
  }
}

int cfo_set_state(cfo_sim *S, const double *state, int broadcast) {
  if (!S || !state) return -1;
  if (!S->have_state) return -3;      /* needs world params from a reset */
  for (int j = 0; j < S->D; ++j)
    for (int64_t i = 0; i < S->MN; ++i) S->x[j * S->MN + i] = broadcast ? state[j] : state[j * S->MN + i];
  rearm_controllers(S);
  return 0;
}

int cfo_set_full(cfo_sim *S, const double *state, const double *ctrl, const double *wparam,
                 const double *mind2, int64_t step_counter) {
  if (!S) return -1;
  if (state) memcpy(S->x, state, sizeof(double) * S->D * S->MN);
  if (ctrl) memcpy(S->ctrl, ctrl, sizeof(double) * 14 * S->MN);
  if (wparam) memcpy(S->wp, wparam, sizeof(double) * S->P * S->M);
  if (mind2) memcpy(S->mind2, mind2, sizeof(double) * 8 * S->MN);
  if (step_counter >= 0) S->s = (uint32_t)step_counter;
  S->have_state = 1;
  return 0;
}

/* teacher forcing of the planning-rollout state (either pointer may be NULL = keep) */
int cfo_set_plan_state(cfo_sim *S, const double *eps, const double *cost_run) {
  if (!S) return -1;
  if (eps) memcpy(S->eps, eps, sizeof(double) * 4 * S->MN);
  if (cost_run) memcpy(S->cost, cost_run, sizeof(double) * S->MN);
  return 0;
}

/* ------------------------------------------------------------------------------------------ */
/* C8: one cf_step call = n_steps physics steps, per drone, in this order:
 *  (1) command fetch  (2) position tick  (3) attitude tick + mixer  (4) disturbance draw
 *  (5) integrate      (6) s += 1         (7) obstacle minima        (8) record */
static int step_impl(cfo_sim *S, const float *cmds, const double *cmds64, int n_cmds, int cmd_hold, int n_steps,
                     int record_every, double *record, size_t record_len);

int cfo_step(cfo_sim *S, const float *cmds, int n_cmds, int cmd_hold, int n_steps, int record_every,
             double *record, size_t record_len) {
  if (!cmds) return -1;
  return step_impl(S, cmds, NULL, n_cmds, cmd_hold, n_steps, record_every, record, record_len);
}

/* The same step with float64 commands [K][MN][4] (CFO_CMD_BUFFER only): used by oracle/grad.py, whose finite
 * differences perturb a command by less than float32 resolves. */
int cfo_step_f64cmd(cfo_sim *S, const double *cmds64, int n_cmds, int cmd_hold, int n_steps) {
  if (!S || !cmds64 || S->p.cmd_source != CFO_CMD_BUFFER) return -1;
  return step_impl(S, NULL, cmds64, n_cmds, cmd_hold, n_steps, 0, NULL, 0);
}

static int step_impl(cfo_sim *S, const float *cmds, const double *cmds64, int n_cmds, int cmd_hold, int n_steps,
                     int record_every, double *record, size_t record_len) {
  if (!S || n_steps < 1 || cmd_hold < 1 || record_every < 0 || (!cmds && !cmds64)) return -1;
  if (!S->have_state) return -3;
  if ((int64_t)n_cmds * cmd_hold < n_steps) return -2;
  const cfo_params *p = &S->p;
  if (p->cmd_source == CFO_CMD_NOMINAL_PLUS_NOISE && p->worlds_per_ctrl > 0 &&
      (S->M - 1) / p->worlds_per_ctrl >= p->n_ctrl) return -2;
  const int D = S->D;
  const int64_t MN = S->MN, N = S->N;
  const uint32_t s0 = S->s;
  const int att_div = (int)(p->f_phys / p->f_att), pos_div = (int)(p->f_phys / p->f_pos);
  const int fp = S->model == CFO_MODEL_FIRST_PRINCIPLES;
  size_t n_rec = 0;
  if (record_every > 0) {
    n_rec = (size_t)((s0 + (uint32_t)n_steps) / (uint32_t)record_every - s0 / (uint32_t)record_every);
    if (n_rec > 0 && (!record || record_len < n_rec * (size_t)D * (size_t)MN)) return -4;
  }
  uint32_t att_ticks = 0, pos_ticks = 0;
  int nthreads = cfo_num_threads();
  (void)nthreads;
#pragma omp parallel for schedule(static) num_threads(nthreads)
  for (int64_t i = 0; i < MN; ++i) {
    const int64_t w = i / N, n = i % N, wg = w + p->world_offset;
    plant_t pl;
    load_plant(S, w, &pl);
    double x[17], c[14], md2[8], cmd[4] = { 0, 0, 0, 0 };
    for (int j = 0; j < D; ++j) x[j] = S->x[j * MN + i];
    for (int j = 0; j < 14; ++j) c[j] = S->ctrl[j * MN + i];
    for (int j = 0; j < 8; ++j) md2[j] = S->mind2[j * MN + i];
    double eps[4], cost = S->cost[i];
    for (int j = 0; j < 4; ++j) eps[j] = S->eps[j * MN + i];
    double *iR = c, *ip = c + 3, *att_cmd = c + 6, *rpm_cmd = c + 10;
    uint32_t s = s0, my_att = 0, my_pos = 0;
    for (int t = 0; t < n_steps; ++t) {
      /* (1) command fetch */
      if (t % cmd_hold == 0) {
        int k = t / cmd_hold;
        if (p->cmd_source == CFO_CMD_BUFFER) {
          for (int j = 0; j < 4; ++j)
            cmd[j] = cmds64 ? cmds64[((size_t)k * MN + i) * 4 + j] : (double)cmds[((size_t)k * MN + i) * 4 + j];
        } else {   /* nominal + sigma .* z, clipped; NOISE stream indexed by the global step */
          uint32_t r[4]; double z[4];
          philox_at(S->seed, wg, n, s, STREAM_NOISE, r);
          cfo_normal_pair(r[0], r[1], &z[0], &z[1]);
          cfo_normal_pair(r[2], r[3], &z[2], &z[3]);
          /* R25: temporally correlated noise, AR(1): eps <- z for the first command after a
           * re-arm, else eps <- beta eps + sqrt(1 - beta^2) z  (stationary, unit variance; beta = 0: white) */
          const int fresh = isnan(eps[0]);
          const double gain = sqrt(1.0 - p->noise_beta * p->noise_beta);
          for (int j = 0; j < 4; ++j) eps[j] = fresh ? z[j] : p->noise_beta * eps[j] + gain * z[j];
          /* R26: one nominal sequence per controller of this shard, controller = local world / worlds_per_ctrl
           * (the noise stays keyed by the GLOBAL world index wg, so a controller's rollouts do not depend on the shard) */
          const int64_t cidx = p->worlds_per_ctrl > 0 ? w / p->worlds_per_ctrl : 0;
          const float *nom = cmds + ((size_t)cidx * (size_t)n_cmds + (size_t)k) * 4;
          for (int j = 0; j < 4; ++j)
            cmd[j] = clipd((double)nom[j] + p->noise_sigma[j] * eps[j], p->cmd_lo[j], p->cmd_hi[j]);
        }
        if (p->iface == CFO_IF_ATTITUDE) for (int j = 0; j < 4; ++j) att_cmd[j] = cmd[j];
        if (p->iface == CFO_IF_ROTOR) for (int j = 0; j < 4; ++j) rpm_cmd[j] = clipd(cmd[j], p->rpm_min, p->rpm_max);
        if (p->iface == CFO_IF_TORQUE) mixer(p, cmd[3], cmd, rpm_cmd);   /* cmd = (tau_x, tau_y, tau_z, F) */
      }
      /* (2) position controller tick */
      if (p->iface == CFO_IF_POSITION && s % (uint32_t)pos_div == 0) {
        double R[3][3];
        if (fp) quat_to_R(x + 3, R); else euler_to_R(x[3], x[4], x[5], R);
        double zB[3] = { R[0][2], R[1][2], R[2][2] };
        cfo_position_tick(p, x, fp ? x + 7 : x + 6, zB, cmd, ip, att_cmd);
        ++my_pos;
      }
      /* (3) attitude controller tick + mixer (first-principles model only) */
      if (fp && p->iface >= CFO_IF_ATTITUDE && s % (uint32_t)att_div == 0) {
        cfo_attitude_tick(p, x + 3, x + 10, att_cmd, iR, NULL, NULL, rpm_cmd);
        ++my_att;
      }
      /* (4) disturbance, held over all RK4 stages */
      double fdist[3] = { 0, 0, 0 };
      if (p->dist_sigma > 0.0) {
        uint32_t r[4]; double z[4];
        philox_at(S->seed, wg, n, s, STREAM_DIST, r);
        cfo_normal_pair(r[0], r[1], &z[0], &z[1]);
        cfo_normal_pair(r[2], r[3], &z[2], &z[3]);
        for (int j = 0; j < 3; ++j) fdist[j] = p->dist_sigma * z[j];
      }
      /* (5) integrate */
      integrate(S, &pl, x, fp ? rpm_cmd : att_cmd, fdist);
      /* (6) */
      s += 1;
      /* (7) obstacle minima with the post-step position (R21) */
      for (int j = 0; j < p->n_obstacles; ++j) {
        double dx_ = x[0] - p->obstacles[j][0], dy_ = x[1] - p->obstacles[j][1], dz_ = x[2] - p->obstacles[j][2];
        double d2 = dx_ * dx_ + dy_ * dy_ + dz_ * dz_;
        if (d2 < md2[j]) md2[j] = d2;
      }
      /* (7b) running rollout cost on the post-step state (R27): h (w_pos |p - goal|^2 + w_vel |v|^2) */
      if (p->cost_on) {
        const double *v = fp ? x + 7 : x + 6;
        double ex = x[0] - p->cost_goal[0], ey = x[1] - p->cost_goal[1], ez = x[2] - p->cost_goal[2];
        cost += (1.0 / p->f_phys) * (p->cost_w_pos * (ex * ex + ey * ey + ez * ez) +
                                     p->cost_w_vel * (v[0] * v[0] + v[1] * v[1] + v[2] * v[2]));
      }
      /* (8) record */
      if (record_every > 0 && s % (uint32_t)record_every == 0) {
        size_t slot = (size_t)(s / (uint32_t)record_every - s0 / (uint32_t)record_every - 1);
        for (int j = 0; j < D; ++j) record[(slot * D + j) * MN + i] = x[j];
        if (i == 0) {
          uint32_t gslot = S->n_rec_total + (uint32_t)slot;
          if (gslot < CFO_REC_TABLE_CAP) S->rec_table[gslot] = s;
        }
      }
    }
    for (int j = 0; j < D; ++j) S->x[j * MN + i] = x[j];
    for (int j = 0; j < 14; ++j) S->ctrl[j * MN + i] = c[j];
    for (int j = 0; j < 8; ++j) S->mind2[j * MN + i] = md2[j];
    for (int j = 0; j < 4; ++j) S->eps[j * MN + i] = eps[j];
    S->cost[i] = cost;
    if (i == 0) { att_ticks = my_att; pos_ticks = my_pos; }
  }
  S->s = s0 + (uint32_t)n_steps;
  S->att_ticks += att_ticks; S->pos_ticks += pos_ticks; S->n_rec_total += (uint32_t)n_rec;
  return 0;
}

int cfo_get_state(cfo_sim *S, double *out) {
  if (!S || !out) return -1;
  memcpy(out, S->x, sizeof(double) * S->D * S->MN);
  return 0;
}

int cfo_get_aux(cfo_sim *S, int which, void *out) {
  if (!S || !out) return -1;
  switch (which) {
    case CFO_AUX_COUNTERS: {
      uint32_t *o = (uint32_t *)out;
      o[0] = S->s; o[1] = S->att_ticks; o[2] = S->pos_ticks; o[3] = S->n_rec_total;
      return 0;
    }
    case CFO_AUX_MIN_DIST: {   /* C10: per world, min over drones, obstacles and steps of |p - c_j| - r_j */
      double *o = (double *)out;
      for (int64_t w = 0; w < S->M; ++w) {
        double best = INFINITY;
        for (int64_t n = 0; n < S->N; ++n)
          for (int j = 0; j < S->p.n_obstacles; ++j) {
            double d = sqrt(S->mind2[j * S->MN + w * S->N + n]) - S->p.obstacles[j][3];
            if (d < best) best = d;
          }
        o[w] = best;
      }
      return 0;
    }
    case CFO_AUX_CTRL: memcpy(out, S->ctrl, sizeof(double) * 14 * S->MN); return 0;
    case CFO_AUX_WORLD_PARAMS: memcpy(out, S->wp, sizeof(double) * S->P * S->M); return 0;
    case CFO_AUX_REC_TABLE: memcpy(out, S->rec_table, sizeof(S->rec_table)); return 0;
    case CFO_AUX_MIN_D2: memcpy(out, S->mind2, sizeof(double) * 8 * S->MN); return 0;
    case CFO_AUX_EPS: memcpy(out, S->eps, sizeof(double) * 4 * S->MN); return 0;
    case CFO_AUX_COST_RUN: memcpy(out, S->cost, sizeof(double) * S->MN); return 0;
    case CFO_AUX_COST: {   /* R27: J = J_run + w_term |p - goal|^2 + w_obs max(0, d_safe - d_min)^2 + w_coll [d_min < 0] */
      double *o = (double *)out;
      const cfo_params *p = &S->p;
      for (int64_t i = 0; i < S->MN; ++i) {
        double ex = S->x[i] - p->cost_goal[0], ey = S->x[S->MN + i] - p->cost_goal[1], ez = S->x[2 * S->MN + i] - p->cost_goal[2];
        double J = S->cost[i] + p->cost_w_term * (ex * ex + ey * ey + ez * ez);
        double dmin = INFINITY;   /* C10 for this drone */
        for (int j = 0; j < p->n_obstacles; ++j) {
          double d = sqrt(S->mind2[j * S->MN + i]) - p->obstacles[j][3];
          if (d < dmin) dmin = d;
        }
        if (dmin < p->cost_d_safe) J += p->cost_w_obs * (p->cost_d_safe - dmin) * (p->cost_d_safe - dmin);
        if (dmin < 0.0) J += p->cost_w_coll;
        o[i] = J;
      }
      return 0;
    }
  }
  return -1;
}
