// cf_rollout_fp.cu -- instantiations of the rollout kernel for the first-principles model.
// Lean instantiations exist for the benchmark configurations; OPT_ALL is the general kernel for everything else.
#include "cf_device.cuh"

namespace cf {

struct EntryFP { int integ, iface, opt; const char *name; void (*fn)(const StepArgs, const DevParams); };

#define CF_FP(INTEG, IFACE, OPT) \
  { INTEG, IFACE, OPT, "rollout<FP," #INTEG "," #IFACE "," #OPT ">", rollout_kernel<MODEL_FP, INTEG, IFACE, OPT> }

static const EntryFP kTableFP[] = {
  // configs[0] / configs[1]: attitude interface, nominal plant
  CF_FP(INTEG_EULER, IF_ATTITUDE, 0),
  CF_FP(INTEG_RK4, IF_ATTITUDE, 0),
  // configs[4] (+5E): domain randomisation + Philox disturbance
  CF_FP(INTEG_EULER, IF_ATTITUDE, OPT_RANDP | OPT_DIST),
  CF_FP(INTEG_RK4, IF_ATTITUDE, OPT_RANDP | OPT_DIST),
  // general kernels
  CF_FP(INTEG_EULER, IF_ROTOR, OPT_ALL),    CF_FP(INTEG_RK4, IF_ROTOR, OPT_ALL),
  CF_FP(INTEG_EULER, IF_TORQUE, OPT_ALL),   CF_FP(INTEG_RK4, IF_TORQUE, OPT_ALL),
  CF_FP(INTEG_EULER, IF_ATTITUDE, OPT_ALL), CF_FP(INTEG_RK4, IF_ATTITUDE, OPT_ALL),
  CF_FP(INTEG_EULER, IF_POSITION, OPT_ALL), CF_FP(INTEG_RK4, IF_POSITION, OPT_ALL),
};

bool launch_fp(int integ, int iface, int opt, const StepArgs *A, const DevParams *P, const LaunchCfg *L,
               const char **name, int *opt_used, bool dry) {
  const EntryFP *best = nullptr;
  for (const EntryFP &e : kTableFP) {
    if (e.integ != integ || e.iface != iface || (e.opt & opt) != opt) continue;
    if (!best || __builtin_popcount(e.opt) < __builtin_popcount(best->opt)) best = &e;
  }
  if (!best) return false;
  if (name) *name = best->name;
  if (opt_used) *opt_used = best->opt;
  if (!dry) best->fn<<<L->grid, L->block, L->smem, L->stream>>>(*A, *P);
  return true;
}

}  // namespace cf
