// cf_rollout_ab.cu -- instantiations of the rollout kernel for the abstracted (identified) model, Eqs. (7)-(10)
// (PAPER.md:L334-L354).
#include "cf_device.cuh"

namespace cf {

#define CF_AB1(INTEG, IFACE, OPT, REC) \
  { INTEG, IFACE, OPT, REC, "rollout<AB," #INTEG "," #IFACE "," #OPT "," #REC ">", rollout_kernel<MODEL_AB, INTEG, IFACE, OPT, REC> }
// a lean configuration: one kernel per record mode
#define CF_AB(INTEG, IFACE, OPT) \
  CF_AB1(INTEG, IFACE, OPT, REC_NONE), CF_AB1(INTEG, IFACE, OPT, REC_SCALAR), CF_AB1(INTEG, IFACE, OPT, REC_TMA)
#define CF_AB_GEN(INTEG, IFACE) CF_AB1(INTEG, IFACE, OPT_ALL, REC_RUNTIME)

static const RolloutEntry kTableAB[] = {
  // configs[2]: planning rollouts, in-kernel nominal + noise commands, obstacle distance, jittered (a,b,c)
  CF_AB(INTEG_EULER, IF_ATTITUDE, OPT_RANDP | OPT_OBST | OPT_NOISE),
  // sampling-based planner: the same rollout + correlated noise + rollout cost
  CF_AB(INTEG_EULER, IF_ATTITUDE, OPT_RANDP | OPT_OBST | OPT_NOISE | OPT_AR | OPT_COST),
  // variant 3B: the same with a command buffer
  CF_AB(INTEG_EULER, IF_ATTITUDE, OPT_RANDP | OPT_OBST),
  // configs[3]: swarm, position interface, per-world mass
  CF_AB(INTEG_EULER, IF_POSITION, OPT_RANDP),
  CF_AB(INTEG_EULER, IF_ATTITUDE, 0),
  // general kernels
  CF_AB_GEN(INTEG_EULER, IF_ATTITUDE), CF_AB_GEN(INTEG_RK4, IF_ATTITUDE),
  CF_AB_GEN(INTEG_EULER, IF_POSITION), CF_AB_GEN(INTEG_RK4, IF_POSITION),
};

bool launch_ab(int integ, int iface, int opt, int rec_mode, const StepArgs *A, const DevParams *P, const LaunchCfg *L,
               const char **name, int *opt_used, bool dry) {
  const RolloutEntry *best = pick_rollout(kTableAB, (int)(sizeof(kTableAB) / sizeof(kTableAB[0])), integ, iface, opt, rec_mode);
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
