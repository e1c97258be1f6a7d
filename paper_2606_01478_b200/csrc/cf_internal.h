// cf_internal.h -- host-side handle shared by the translation units of libcf.so (cf_api.cu, cf_mppi.cu).  Not installed.
#pragma once
#include "../../include/cf.h"
#include "cf_device.cuh"

#include <cstdarg>
#include <cstdio>

using cf::Counters; using cf::DevParams;

struct cf_sim {
  long long M, N, MN;
  int model, D, P;
  cf_params p;
  DevParams dp;
  int opt;                    // option bits this configuration needs
  // workspace carving (device pointers into the caller's buffer)
  float *state, *ctrl, *wparam, *min_d2;
  float *bcast_buf;           // [D] pending broadcast state (cf_set_state(broadcast) is folded into the next cf_step)
  float *md_drone;            // [MN] per-drone minimum distance written by the rollout kernel's epilogue
  float *eps;                 // [4][MN] AR(1) command-noise state (noise mode with noise_beta != 0), else nullptr
  float *cost_run, *cost_drone;   // [MN] running / total rollout cost (cost_on), else nullptr
  bool cost_valid;            // cost_drone holds the cost of the current state
  // the last cf_step call, for cf_mppi_update: did it start from a fresh re-arm, where, and with which commands
  bool rearmed;               // no cf_step since the last cf_reset / cf_set_state
  bool last_fresh; long long last_s0; int last_n_steps, last_n_cmds, last_cmd_hold;
  bool pending_bcast, md_valid;
  int last_rec_mode;          // record mode of the last cf_step launch (cf_describe_launch names that kernel)
  bool last_rec_heavy;        // ... and whether it took the large blocks of record-every-step runs
  Counters *counters;
  uint32_t *rec_table;
  cudaStream_t stream;
  uint64_t seed;
  long long s_host;           // host mirror of the step counter
  long long n_rec_host;
  bool have_state;
  float hover_rpm;
  // cf_rollout_host: a second stream for the result copies and one event per slice (created on first use)
  bool wparam_foreign = false;   // cf_set_full replaced the parameter planes (cf_reset re-draws them and clears this)
  cudaStream_t copy_stream = nullptr;
  bool force_general = false;     // CF_FORCE_GENERAL=1 at cf_create: dispatch the general kernel everywhere (measurement)
  bool copy_stream_owned = false; // created by cf_rollout_host (destroyed with the handle) vs given by cf_set_copy_stream
  cudaEvent_t slice_ev[16] = {};
};

int cf_materialise(cf_sim *sim);         // cf_api.cu: write a pending broadcast cf_set_state into the planes
int cf_refresh_cost(cf_sim *sim);        // cf_api.cu: cost_drone <- J of the current planes
char *cf_err_buf();                      // thread-local, 512 bytes (cf_api.cu)
inline int fail(int code, const char *fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(cf_err_buf(), 512, fmt, ap);
  va_end(ap);
  return code;
}
#define CF_CUDA(expr) do { cudaError_t e_ = (expr); if (e_ != cudaSuccess) \
  return fail(CF_E_CUDA, "%s: %s", #expr, cudaGetErrorString(e_)); } while (0)

