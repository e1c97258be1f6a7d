// cf_rollout_ab.cu -- instantiations of the rollout kernel for the abstracted (identified) model, Eqs. (7)-(10)
// (PAPER.md:L334-L354).
#include "cf_device.cuh"

namespace cf {

struct EntryAB { int integ, iface, opt; const char *name; void (*fn)(const StepArgs, const DevParams); };

#define CF_AB(INTEG, IFACE, OPT) \
  { INTEG, IFACE, OPT, "rollout<AB," #INTEG "," #IFACE "," #OPT ">", rollout_kernel<MODEL_AB, INTEG, IFACE, OPT> }

static const EntryAB kTableAB[] = {
  // configs[2]: planning rollouts, in-kernel nominal + noise commands, obstacle distance, jittered (a,b,c)
  CF_AB(INTEG_EULER, IF_ATTITUDE, OPT_RANDP | OPT_OBST | OPT_NOISE),
  // sampling-based planner: the same rollout + correlated noise + rollout cost
  CF_AB(INTEG_EULER, IF_ATTITUDE, OPT_RANDP | OPT_OBST | OPT_NOISE | OPT_COST),
  // variant 3B: the same with a command buffer
  CF_AB(INTEG_EULER, IF_ATTITUDE, OPT_RANDP | OPT_OBST),
  // configs[3]: swarm, position interface, per-world mass
  CF_AB(INTEG_EULER, IF_POSITION, OPT_RANDP),
  CF_AB(INTEG_EULER, IF_ATTITUDE, 0),
  // general kernels
  CF_AB(INTEG_EULER, IF_ATTITUDE, OPT_ALL), CF_AB(INTEG_RK4, IF_ATTITUDE, OPT_ALL),
  CF_AB(INTEG_EULER, IF_POSITION, OPT_ALL), CF_AB(INTEG_RK4, IF_POSITION, OPT_ALL),
};

bool launch_ab(int integ, int iface, int opt, const StepArgs *A, const DevParams *P, const LaunchCfg *L,
               const char **name, int *opt_used, bool dry) {
  const EntryAB *best = nullptr;
  for (const EntryAB &e : kTableAB) {
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
