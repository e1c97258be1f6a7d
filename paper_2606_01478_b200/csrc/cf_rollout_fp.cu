// cf_rollout_fp.cu -- instantiations of the rollout kernel for the first-principles model.
// Lean instantiations exist for the benchmark configurations; OPT_ALL is the general kernel for everything else.
#include "cf_device.cuh"

namespace cf {

#define CF_FP1(INTEG, IFACE, OPT, REC) \
  { INTEG, IFACE, OPT, REC, "rollout<FP," #INTEG "," #IFACE "," #OPT "," #REC ">", rollout_kernel<MODEL_FP, INTEG, IFACE, OPT, REC> }
#define CF_FP(INTEG, IFACE, OPT) \
  CF_FP1(INTEG, IFACE, OPT, REC_NONE), CF_FP1(INTEG, IFACE, OPT, REC_SCALAR), CF_FP1(INTEG, IFACE, OPT, REC_TMA)
#define CF_FP_GEN(INTEG, IFACE) CF_FP1(INTEG, IFACE, OPT_ALL, REC_RUNTIME)

static const RolloutEntry kTableFP[] = {
  // configs[0] / configs[1]: attitude interface, nominal plant
  CF_FP(INTEG_EULER, IF_ATTITUDE, 0),
  CF_FP(INTEG_RK4, IF_ATTITUDE, 0),
  // configs[4] (+5E): domain randomisation + Philox disturbance
  CF_FP(INTEG_EULER, IF_ATTITUDE, OPT_RANDP | OPT_DIST),
  CF_FP(INTEG_RK4, IF_ATTITUDE, OPT_RANDP | OPT_DIST),
  // record-every-step runs with the pair schedule as a compile-time fact (REC_PAIR, cf_device.cuh)
  // (RK4 only: configs[4] 1.288 -> 1.253 ms; the Euler kernel of variant 5E measured 2.8 % slower with it)
  CF_FP1(INTEG_RK4, IF_ATTITUDE, 0, REC_PAIR), CF_FP1(INTEG_RK4, IF_ATTITUDE, OPT_RANDP | OPT_DIST, REC_PAIR),
  // the pair-written loop for the other record modes (REC_*_P): configs[0], configs[1], the world-count sweep
  CF_FP1(INTEG_RK4, IF_ATTITUDE, 0, REC_NONE_P), CF_FP1(INTEG_RK4, IF_ATTITUDE, 0, REC_SCALAR_P), CF_FP1(INTEG_RK4, IF_ATTITUDE, 0, REC_TMA_P),
  CF_FP1(INTEG_EULER, IF_ATTITUDE, 0, REC_NONE_P), CF_FP1(INTEG_EULER, IF_ATTITUDE, 0, REC_SCALAR_P), CF_FP1(INTEG_EULER, IF_ATTITUDE, 0, REC_TMA_P),
  // round 3 ("dynamically select only the required functions", L282 "direct rotor velocity" control, L330 the
  // full Mellinger stack): the nominal plant behind the rotor interface (motor-level control) and behind the position
  // interface (position controller -> attitude controller -> mixer), which until now fell to the general kernel
  CF_FP(INTEG_RK4, IF_ROTOR, 0), CF_FP(INTEG_EULER, IF_ROTOR, 0),
  CF_FP(INTEG_RK4, IF_POSITION, 0), CF_FP(INTEG_EULER, IF_POSITION, 0),
  // general kernels
  CF_FP_GEN(INTEG_EULER, IF_ROTOR),    CF_FP_GEN(INTEG_RK4, IF_ROTOR),
  CF_FP_GEN(INTEG_EULER, IF_TORQUE),   CF_FP_GEN(INTEG_RK4, IF_TORQUE),
  CF_FP_GEN(INTEG_EULER, IF_ATTITUDE), CF_FP_GEN(INTEG_RK4, IF_ATTITUDE),
  CF_FP_GEN(INTEG_EULER, IF_POSITION), CF_FP_GEN(INTEG_RK4, IF_POSITION),
};

bool launch_fp(int integ, int iface, int opt, int rec_mode, const StepArgs *A, const DevParams *P, const LaunchCfg *L,
               const char **name, int *opt_used, bool dry) {
  const RolloutEntry *best = pick_rollout(kTableFP, (int)(sizeof(kTableFP) / sizeof(kTableFP[0])), integ, iface, opt, rec_mode);
  if (!best) return false;
  if (name) *name = best->name;
  if (opt_used) *opt_used = best->opt;
  if (!dry) {
    if (L->smem > 48 * 1024) cudaFuncSetAttribute(best->fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)L->smem);
    best->fn<<<L->grid, L->block, L->smem, L->stream>>>(*A, *P);
  }
  return true;
}

}  // namespace cf
