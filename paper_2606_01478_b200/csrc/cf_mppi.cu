// cf_mppi.cu -- the sampling-based planner's update step (hybrid iCEM / MPPI; readings R28-R32 in
// DESIGN.md): per controller, exact top-n_elite selection of the rollout costs, exponential weighting, weighted mean of
// the elites' command sequences (regenerated from the Philox counters -- the 500 k x H sampled commands are never
// stored), controller score; then the best controller's plan and the warm-started nominal sequences.
//
// One thread-block CLUSTER of 8 CTAs per controller does everything for its K_c rollouts (K_c = 100 000 costs = 400 kB,
// L2 resident); CTA r of the cluster owns the contiguous slice [r S, (r+1) S) of the costs.  The CTAs exchange
// histograms, counts and partial sums through distributed shared memory (cluster.map_shared_rank) between
// cluster barriers -- no global atomics, no extra launches:
//   1. radix select (4 passes x 8 bits, MSB first) of the n_elite-th smallest cost key -> threshold key T and the number
//      r of keys equal to T that are admitted (ties go to the lowest world index, R28); per-CTA shared-memory histograms
//      (warp-aggregated atomics, double-buffered so one cluster barrier per pass suffices), summed by every CTA;
//   2. ordered compaction of the elites: per-CTA counts exchanged over DSMEM + one block scan over per-thread segment
//      counts -> ascending index list;
//   3. one thread per elite (spread over the 8 CTAs): weight, regenerate eps / commands for the H knots with the
//      rollout kernel's own arithmetic (bit-identical commands), write w * u rows to scratch;
//   4. fixed-order column sums (per CTA, then over the 8 CTAs in rank order: deterministic), mean, score;
//   5. the last cluster to finish picks the best controller, writes the plan and shifts the nominal sequences.
#include "cf_internal.h"

#include <cmath>
#include <cooperative_groups.h>
#include <mutex>

namespace cg = cooperative_groups;

using namespace cf;

namespace {

constexpr int kThreads = 1024;
constexpr int kCluster = 8;      // CTAs per controller (portable cluster size)
constexpr int kRegKeys = 16;     // cost keys a thread keeps in registers

struct MppiArgs {
  const float *cost;        // [n_ctrl][K_c] rollout costs (world order)
  float4 *nominal;          // [n_ctrl][H] in / out
  float4 *plan;             // [H]
  float *info;              // CF_MPPI_INFO_WORDS
  int32_t *elite_out;       // [n_ctrl][n_elite] or nullptr
  int32_t *elite_idx;       // scratch [n_ctrl][n_elite]
  float4 *rows;             // scratch [n_ctrl][n_elite][H + 1]: w * u[t] (t < H), then (w, w J, 0, 0)
  float4 *mean;             // scratch [n_ctrl][H]
  unsigned int *done;       // scratch, zeroed before the launch
  long long K_c, world0;    // rollouts per controller; global index of this shard's world 0
  int n_ctrl, H, hold, n_elite, shift;
  float inv_lambda;
  uint32_t s_start;         // step at which the rollouts formed their first command
  uint32_t rk[20];          // Philox round keys of the simulator's seed
};

// R28: uint32 key whose unsigned order is the IEEE total order of the float32 cost, NaN (either sign) last
__device__ __forceinline__ uint32_t cost_key(float c) {
  uint32_t b = __float_as_uint(c);
  if (c != c) return 0xFFFFFFFFu;
  return (b & 0x80000000u) ? ~b : (b | 0x80000000u);
}
__device__ __forceinline__ float key_cost(uint32_t k) {
  return __uint_as_float((k & 0x80000000u) ? (k & 0x7FFFFFFFu) : ~k);
}

// exclusive block scan of one unsigned per thread (1024 threads); returns the exclusive prefix, *total = block sum
__device__ __forceinline__ unsigned block_exscan(unsigned v, unsigned *warp_sums, unsigned *total) {
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  unsigned inc = v;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) { unsigned t = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= o) inc += t; }
  if (lane == 31) warp_sums[wid] = inc;
  __syncthreads();
  if (wid == 0) {
    unsigned s = warp_sums[lane], si = s;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { unsigned t = __shfl_up_sync(0xffffffffu, si, o); if (lane >= o) si += t; }
    warp_sums[lane] = si - s;                 // exclusive warp offsets
    if (lane == 31) warp_sums[32] = si;
  }
  __syncthreads();
  unsigned ex = warp_sums[wid] + inc - v;
  *total = warp_sums[32];
  __syncthreads();                            // warp_sums may be reused by the caller
  return ex;
}

// what a CTA publishes to the other CTAs of its cluster (read through DSMEM)
struct Shared {
  unsigned hist[2][256];      // radix-pass histogram of this CTA's slice, double-buffered over passes
  unsigned n_less, n_eq;      // keys below / equal to the threshold in this CTA's slice
  uint32_t kmin;              // smallest key of the slice
  float colsum[kThreads];     // this CTA's partial column sums (first 4 (H + 1) entries)
};

__global__ void __cluster_dims__(kCluster, 1, 1) __launch_bounds__(kThreads, 1)
mppi_update_kernel(const __grid_constant__ MppiArgs A, const __grid_constant__ DevParams P) {
  __shared__ Shared sh;
  __shared__ unsigned tot[256];
  __shared__ unsigned warp_sums[33];
  __shared__ unsigned sh_prefix, sh_rank;
  __shared__ float sh_part[kThreads];
  __shared__ float sh_sum[2];
  __shared__ bool is_last;
  cg::cluster_group cluster = cg::this_cluster();
  const int c = blockIdx.x / kCluster, rk = (int)cluster.block_rank();
  const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
  const long long K = A.K_c;
  const float *cost = A.cost + (long long)c * K;
  // slice of this CTA: S keys (a multiple of kThreads so that thread segments tile it exactly)
  const long long S = ((K + kCluster - 1) / kCluster + kThreads - 1) / kThreads * kThreads;
  const long long s_lo = (long long)rk * S < K ? (long long)rk * S : K;
  const long long s_hi = s_lo + S < K ? s_lo + S : K;

  // thread t owns the contiguous segment [lo, hi) of the slice.  Its first kRegKeys keys are read ONCE (all loads in
  // flight together) and stay in registers for the four radix passes and the compaction; a longer segment (more than
  // kCluster * kThreads * kRegKeys = 131 072 rollouts per controller) re-reads its tail from L2 in every pass.
  const long long seg = S / kThreads;
  const long long lo = s_lo + (long long)tid * seg < s_hi ? s_lo + (long long)tid * seg : s_hi;
  const long long hi = lo + seg < s_hi ? lo + seg : s_hi;
  const int n_reg = (int)(hi - lo < kRegKeys ? hi - lo : kRegKeys);
  uint32_t keys[kRegKeys];
#pragma unroll
  for (int j = 0; j < kRegKeys; ++j) keys[j] = j < n_reg ? cost_key(__ldg(cost + lo + j)) : 0xFFFFFFFFu;

  // ---- 1. radix select of the n_elite-th smallest key ---------------------------------------------------------
  uint32_t prefix = 0, mask = 0;
  unsigned rank = (unsigned)A.n_elite;        // 1-based rank inside the current candidate set
  for (int pass = 0; pass < 4; ++pass) {
    const int shf = 24 - 8 * pass, buf = pass & 1;
    if (tid < 256) sh.hist[buf][tid] = 0;     // last read by the other CTAs two passes ago (a cluster barrier since)
    __syncthreads();
    auto count = [&](bool valid, uint32_t k) {
      unsigned bin = (valid && (k & mask) == prefix) ? (k >> shf) & 255u : 256u;
      unsigned peers = __match_any_sync(0xffffffffu, bin);            // warp-aggregated shared-memory atomics
      if (bin < 256 && lane == __ffs(peers) - 1) atomicAdd(&sh.hist[buf][bin], (unsigned)__popc(peers));
    };
#pragma unroll
    for (int j = 0; j < kRegKeys; ++j) count(j < n_reg, keys[j]);
    for (long long j = kRegKeys; j < seg; ++j) {                      // (uniform trip count: warp-collective inside)
      bool valid = lo + j < hi;
      count(valid, valid ? cost_key(__ldg(cost + lo + j)) : 0u);
    }
    cluster.sync();                                                   // every CTA's histogram is complete
    if (tid < 256) {                                                  // every CTA sums all 8 (same result everywhere)
      unsigned s = 0;
#pragma unroll
      for (int r = 0; r < kCluster; ++r) s += cluster.map_shared_rank(&sh, r)->hist[buf][tid];
      tot[tid] = s;
    }
    __syncthreads();
    if (wid == 0) {                                                   // find the bucket that holds the rank
      unsigned cnt[8], sum = 0;
#pragma unroll
      for (int j = 0; j < 8; ++j) { cnt[j] = tot[lane * 8 + j]; sum += cnt[j]; }
      unsigned inc = sum;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) { unsigned t = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= o) inc += t; }
      unsigned below = inc - sum;                                     // keys in lower lanes' buckets
      if (rank > below && rank <= inc) {                              // exactly one lane
        unsigned r = rank - below;
#pragma unroll
        for (int j = 0; j < 8; ++j) {
          if (r != 0 && r <= cnt[j]) { sh_prefix = prefix | ((uint32_t)(lane * 8 + j) << shf); sh_rank = r; r = 0; }
          else if (r != 0) r -= cnt[j];
        }
      }
    }
    __syncthreads();
    prefix = sh_prefix; rank = sh_rank; mask |= 0xFFu << shf;
    __syncthreads();
  }
  const uint32_t T = prefix;                  // threshold key; `rank` of the keys equal to T are admitted (lowest indices)

  // ---- 2. ordered compaction: thread t owns the contiguous segment [s_lo + t seg, s_lo + (t+1) seg) ---------------
  unsigned n_less = 0, n_eq = 0;
  uint32_t kmin = 0xFFFFFFFFu;
#pragma unroll
  for (int j = 0; j < kRegKeys; ++j) {
    if (j < n_reg) { uint32_t k = keys[j]; n_less += k < T; n_eq += k == T; kmin = k < kmin ? k : kmin; }
  }
  for (long long i = lo + kRegKeys; i < hi; ++i) {
    uint32_t k = cost_key(__ldg(cost + i));
    n_less += k < T; n_eq += k == T; kmin = k < kmin ? k : kmin;
  }
  unsigned tot_less, tot_eq;
  unsigned ex_less = block_exscan(n_less, warp_sums, &tot_less);
  unsigned ex_eq = block_exscan(n_eq, warp_sums, &tot_eq);
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) { uint32_t t = __shfl_xor_sync(0xffffffffu, kmin, o); kmin = t < kmin ? t : kmin; }
  if (lane == 0) warp_sums[wid] = kmin;
  __syncthreads();
  if (wid == 0) {
    kmin = warp_sums[lane];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) { uint32_t t = __shfl_xor_sync(0xffffffffu, kmin, o); kmin = t < kmin ? t : kmin; }
    if (lane == 0) { sh.n_less = tot_less; sh.n_eq = tot_eq; sh.kmin = kmin; }
  }
  cluster.sync();                                                     // counts and minima of all slices are published
  unsigned less_before = 0, eq_before = 0;
  uint32_t kmin_all = 0xFFFFFFFFu;
#pragma unroll
  for (int r = 0; r < kCluster; ++r) {
    const Shared *o = cluster.map_shared_rank(&sh, r);
    unsigned nl = o->n_less, ne = o->n_eq; uint32_t km = o->kmin;
    if (r < rk) { less_before += nl; eq_before += ne; }
    kmin_all = km < kmin_all ? km : kmin_all;
  }
  const float J_min = key_cost(kmin_all);     // the best rollout is always an elite
  int32_t *eidx = A.elite_idx + (long long)c * A.n_elite;
  {
    unsigned eq_seen = eq_before + ex_eq;
    unsigned pos = less_before + ex_less + (eq_seen < rank ? eq_seen : rank);
    auto admit = [&](long long i, uint32_t k) {
      bool take = k < T || (k == T && eq_seen < rank);
      eq_seen += k == T;
      if (take) {
        eidx[pos] = (int32_t)i;
        if (A.elite_out) A.elite_out[(long long)c * A.n_elite + pos] = (int32_t)i;
        ++pos;
      }
    };
#pragma unroll
    for (int j = 0; j < kRegKeys; ++j) if (j < n_reg) admit(lo + j, keys[j]);
    for (long long i = lo + kRegKeys; i < hi; ++i) admit(i, cost_key(__ldg(cost + i)));
  }
  __threadfence();
  cluster.sync();                                                     // the elite list (written by all 8 CTAs) is complete

  // ---- 3. one thread per elite: weight, regenerated commands (R25, R26 with the rollout kernel's arithmetic) -----
  const int H = A.H, RW = H + 1;
  float4 *rows = A.rows + (long long)c * A.n_elite * RW;
  const float4 *nom = A.nominal + (long long)c * H;
  const int E = (A.n_elite + kCluster - 1) / kCluster;                // elites per CTA
  const int e_lo = rk * E < A.n_elite ? rk * E : A.n_elite, e_hi = e_lo + E < A.n_elite ? e_lo + E : A.n_elite;
  for (int e = e_lo + tid; e < e_hi; e += kThreads) {
    const int k = __ldcg(eidx + e);
    const float J = __ldg(cost + k);
    const float w = expf(-(J - J_min) * A.inv_lambda);                // R29
    const uint32_t wg = (uint32_t)(A.world0 + (long long)c * K + k);
    float eps[4] = { 0, 0, 0, 0 };
    for (int t = 0; t < H; ++t) {
      uint32_t r[4]; float z[4];
      philox4x32_10_rk(A.rk, wg, 0u, A.s_start + (uint32_t)(t * A.hold), STREAM_NOISE, r);
      normal_pair(r[0], r[1], z[0], z[1]);
      normal_pair(r[2], r[3], z[2], z[3]);
      if (P.noise_beta != 0.0f) {
#pragma unroll
        for (int j = 0; j < 4; ++j) { eps[j] = t == 0 ? z[j] : fmaf(P.noise_beta, eps[j], P.noise_gain * z[j]); z[j] = eps[j]; }
      }
      const float4 n4 = __ldg(nom + t);
      const float nv[4] = { n4.x, n4.y, n4.z, n4.w };
      float u[4];
#pragma unroll
      for (int j = 0; j < 4; ++j) u[j] = clipf(fmaf(P.noise_sigma[j], z[j], nv[j]), P.cmd_lo[j], P.cmd_hi[j]);
      rows[(long long)e * RW + t] = make_float4(w * u[0], w * u[1], w * u[2], w * u[3]);
    }
    rows[(long long)e * RW + H] = make_float4(w, w * J, 0.f, 0.f);
  }
  __threadfence_block();
  __syncthreads();

  // ---- 4. deterministic column sums: per CTA (column j of 4 RW, partial p sums its elites p, p + NP, ... in order),
  //         then over the 8 CTAs in rank order by the cluster's CTA 0 ---------------------------------------------------
  const int ncol = 4 * RW, NP = kThreads / ncol;                     // host guarantees ncol <= kThreads
  const float *rowsf = reinterpret_cast<const float *>(rows);
  if (tid < NP * ncol) {
    const int j = tid % ncol, p = tid / ncol;
    float s = 0.f;
#pragma unroll 4
    for (int e = e_lo + p; e < e_hi; e += NP) s += __ldcg(rowsf + (long long)e * ncol + j);
    sh_part[tid] = s;
  }
  __syncthreads();
  if (tid < ncol) {
    float s = 0.f;
    for (int p = 0; p < NP; ++p) s += sh_part[p * ncol + tid];
    sh.colsum[tid] = s;
  }
  cluster.sync();                                                     // all 8 partial column sums are published
  if (rk == 0) {
    float colsum = 0.f;
    if (tid < ncol) {
#pragma unroll
      for (int r = 0; r < kCluster; ++r) colsum += cluster.map_shared_rank(&sh, r)->colsum[tid];
      if (tid == 4 * H) sh_sum[0] = colsum;                           // sum of weights
      if (tid == 4 * H + 1) sh_sum[1] = colsum;                       // sum of w J
    }
    __syncthreads();
    if (tid < 4 * H) reinterpret_cast<float *>(A.mean + (long long)c * H)[tid] = colsum / sh_sum[0];      // R30
    if (tid == 0) {
      A.info[4 * c + 0] = sh_sum[1] / sh_sum[0];                      // R31 score
      A.info[4 * c + 1] = J_min;
      A.info[4 * c + 2] = sh_sum[0];
      A.info[4 * c + 3] = key_cost(T);
    }
  }
  cluster.sync();                             // nobody leaves while CTA 0 may still read its shared memory
  if (rk != 0) return;

  // ---- 5. last cluster: best controller, plan, warm start (R31, R32) ---------------------------------------------
  __threadfence();
  __syncthreads();
  if (tid == 0) is_last = atomicAdd(A.done, 1u) == (unsigned)A.n_ctrl - 1;
  __syncthreads();
  if (!is_last) return;
  __threadfence();
  int best = 0;
  float best_s = __ldcg(A.info + 0);
  for (int cc = 1; cc < A.n_ctrl; ++cc) {
    float s = __ldcg(A.info + 4 * cc);
    if (s < best_s) { best_s = s; best = cc; }
  }
  if (tid == 0) reinterpret_cast<int32_t *>(A.info)[4 * A.n_ctrl] = best;
  for (int t = tid; t < H; t += kThreads) A.plan[t] = __ldcg(A.mean + (long long)best * H + t);
  for (int idx = tid; idx < A.n_ctrl * H; idx += kThreads) {
    int cc = idx / H, t = idx - cc * H, src = t + A.shift < H ? t + A.shift : H - 1;
    A.nominal[idx] = __ldcg(A.mean + (long long)cc * H + src);
  }
}

size_t a256(size_t n) { return (n + 255) & ~(size_t)255; }
struct Scratch { size_t elite_idx, rows, mean, done, total; };
Scratch carve_scratch(int n_ctrl, int n_elite, int H) {
  Scratch s; size_t off = 0;
  s.elite_idx = off; off += a256(sizeof(int32_t) * (size_t)n_ctrl * n_elite);
  s.rows = off;      off += a256(sizeof(float4) * (size_t)n_ctrl * n_elite * (H + 1));
  s.mean = off;      off += a256(sizeof(float4) * (size_t)n_ctrl * H);
  s.done = off;      off += 256;
  s.total = off;
  return s;
}

// ---- the cross-shard selection (reading R31 across ranks) -----------------------------------------------------------------
// row = [score of the shard's best controller, its GLOBAL controller index, plan (H float4)]
__global__ void pack_best_kernel(const float *info, const float4 *plan, int n_ctrl, int H, int ctrl_offset, float *row) {
  const int best = __float_as_int(info[4 * n_ctrl]);
  if (threadIdx.x == 0) { row[0] = info[4 * best]; row[1] = (float)(best + ctrl_offset); }
  for (int t = threadIdx.x; t < 4 * H; t += blockDim.x) row[2 + t] = reinterpret_cast<const float *>(plan)[t];
}
// the row with the smallest (score as a float32 in IEEE total order with NaN last -- the cost_key order --, global
// controller index): identical on every rank whatever the order the rows were gathered in
__global__ void select_row_kernel(const float *rows, int n_rows, int H, float *best_row) {
  __shared__ int win;
  const int W = 2 + 4 * H;
  if (threadIdx.x == 0) {
    int w = 0;
    uint32_t kw = cost_key(rows[0]);
    float iw = rows[1];
    for (int r = 1; r < n_rows; ++r) {
      const uint32_t k = cost_key(rows[(size_t)r * W]);
      const float idx = rows[(size_t)r * W + 1];
      if (k < kw || (k == kw && idx < iw)) { w = r; kw = k; iw = idx; }
    }
    win = w;
  }
  __syncthreads();
  for (int t = threadIdx.x; t < W; t += blockDim.x) best_row[t] = rows[(size_t)win * W + t];
}

int check(const cf_sim *sim, const cf_mppi_params *mp) {
  if (!sim || !mp) return fail(CF_E_ARG, "NULL argument");
  if (mp->struct_size != sizeof(cf_mppi_params)) return fail(CF_E_ARG, "cf_mppi_params.struct_size mismatch");
  const cf_params &p = sim->p;
  if (sim->N != 1 || p.cmd_source != CF_CMD_NOMINAL_PLUS_NOISE || !p.cost_on)
    return fail(CF_E_UNSUPPORTED, "the planner needs N == 1, CF_CMD_NOMINAL_PLUS_NOISE and cost_on");
  if (p.worlds_per_ctrl < 1 || sim->M != (long long)p.n_ctrl * p.worlds_per_ctrl)
    return fail(CF_E_SHAPE, "M must equal n_ctrl * worlds_per_ctrl");
  if (mp->horizon < 1 || mp->cmd_hold < 1 || 4 * (mp->horizon + 1) > kThreads) return fail(CF_E_ARG, "horizon out of range (1..255)");
  if (mp->n_elite < 1 || mp->n_elite > p.worlds_per_ctrl || mp->n_elite > 4096) return fail(CF_E_ARG, "n_elite out of range");
  if (mp->shift < 0 || mp->shift > mp->horizon) return fail(CF_E_ARG, "shift out of range");
  if (!(mp->lambda > 0.f)) return fail(CF_E_ARG, "lambda must be > 0");
  return CF_OK;
}

}  // namespace

extern "C" size_t cf_mppi_scratch_bytes(const cf_sim *sim, const cf_mppi_params *mp) {
  if (check(sim, mp) != CF_OK) return 0;
  return carve_scratch(sim->p.n_ctrl, mp->n_elite, mp->horizon).total;
}

extern "C" int cf_mppi_update(cf_sim *sim, const cf_mppi_params *mp, void *nominal_dev, void *plan_dev, void *info_dev,
                              int32_t *elite_idx_dev, void *scratch_dev, size_t scratch_bytes) {
  int rc = check(sim, mp);
  if (rc != CF_OK) return rc;
  if (!nominal_dev || !plan_dev || !info_dev || !scratch_dev) return fail(CF_E_ARG, "NULL argument");
  if (((uintptr_t)nominal_dev & 15) || ((uintptr_t)plan_dev & 15) || ((uintptr_t)scratch_dev & 255))
    return fail(CF_E_BUFFER, "nominal / plan must be 16-byte, scratch 256-byte aligned");
  Scratch sc = carve_scratch(sim->p.n_ctrl, mp->n_elite, mp->horizon);
  if (scratch_bytes < sc.total) return fail(CF_E_BUFFER, "scratch too small: %zu < %zu", scratch_bytes, sc.total);
  if (!sim->last_fresh || sim->last_n_steps != mp->horizon * mp->cmd_hold ||
      sim->last_n_cmds != mp->horizon || sim->last_cmd_hold != mp->cmd_hold)
    return fail(CF_E_STATE, "cf_mppi_update needs a reset / cf_set_state followed by ONE cf_step of horizon * cmd_hold "
                            "steps with n_cmds == horizon");
  rc = cf_refresh_cost(sim);        // no-op straight after the rollout
  if (rc != CF_OK) return rc;
  MppiArgs A;
  char *base = (char *)scratch_dev;
  A.cost = sim->cost_drone; A.nominal = (float4 *)nominal_dev; A.plan = (float4 *)plan_dev; A.info = (float *)info_dev;
  A.elite_out = elite_idx_dev; A.elite_idx = (int32_t *)(base + sc.elite_idx); A.rows = (float4 *)(base + sc.rows);
  A.mean = (float4 *)(base + sc.mean); A.done = (unsigned int *)(base + sc.done);
  A.K_c = sim->p.worlds_per_ctrl; A.world0 = sim->p.world_offset;
  A.n_ctrl = sim->p.n_ctrl; A.H = mp->horizon; A.hold = mp->cmd_hold; A.n_elite = mp->n_elite; A.shift = mp->shift;
  A.inv_lambda = 1.0f / mp->lambda;
  A.s_start = (uint32_t)sim->last_s0;
  const uint32_t lo = (uint32_t)(sim->seed & 0xFFFFFFFFu), hi = (uint32_t)(sim->seed >> 32);
  for (int r = 0; r < 10; ++r) { A.rk[2 * r] = lo + (uint32_t)r * 0x9E3779B9u; A.rk[2 * r + 1] = hi + (uint32_t)r * 0xBB67AE85u; }
  CF_CUDA(cudaMemsetAsync(A.done, 0, sizeof(unsigned int), sim->stream));
  mppi_update_kernel<<<A.n_ctrl * kCluster, kThreads, 0, sim->stream>>>(A, sim->dp);     // one 8-CTA cluster per controller
  CF_CUDA(cudaGetLastError());
  return CF_OK;
}

// ---- cf_mppi_update_static: the same update with the scratch inside the library (include/cf.h says who needs this) --------
// The array is ordinary global memory of every device that loads this module; it is never freed and never initialised.
// In HOST code the identifier below is only a handle for the runtime's symbol table -- not a device address: handing
// `g_static_scratch` itself to a kernel would make the kernel dereference a host pointer.  The device address is what
// cudaGetSymbolAddress returns, and it differs from device to device, hence the per-device table.
namespace {
static __device__ __align__(256) unsigned char g_static_scratch[CF_MPPI_STATIC_SCRATCH_BYTES];
constexpr int kMaxDevices = 64;
std::mutex g_static_mu;
void *g_static_addr[kMaxDevices] = {};        // device ordinal -> device address of g_static_scratch, filled on first use

// Address of the scratch array on the CURRENT device (looked up once per device, under a lock: callers may be threads).
int static_scratch_addr(int dev, void **out) {
  if (dev < 0 || dev >= kMaxDevices) return fail(CF_E_UNSUPPORTED, "device ordinal %d beyond the %d this table holds", dev, kMaxDevices);
  std::lock_guard<std::mutex> lock(g_static_mu);
  if (!g_static_addr[dev]) {
    void *addr = nullptr;
    CF_CUDA(cudaGetSymbolAddress(&addr, g_static_scratch));      // resolves against the current device's copy of the module
    if (!addr) return fail(CF_E_CUDA, "cudaGetSymbolAddress returned a NULL address for the static scratch");
    g_static_addr[dev] = addr;
  }
  *out = g_static_addr[dev];
  return CF_OK;
}
}  // namespace

extern "C" int cf_mppi_update_static(cf_sim *sim, const cf_mppi_params *mp, void *nominal_dev, void *plan_dev,
                                     void *info_dev, int32_t *elite_idx_dev) {
  int rc = check(sim, mp);
  if (rc != CF_OK) return rc;
  const size_t need = carve_scratch(sim->p.n_ctrl, mp->n_elite, mp->horizon).total;
  if (need > CF_MPPI_STATIC_SCRATCH_BYTES)
    return fail(CF_E_BUFFER, "cf_mppi_update_static: n_ctrl = %d, n_elite = %d, horizon = %d need %zu bytes of scratch, the "
                "built-in array holds %zu; use cf_mppi_update with caller-owned scratch",
                sim->p.n_ctrl, mp->n_elite, mp->horizon, need, (size_t)CF_MPPI_STATIC_SCRATCH_BYTES);
  // the address is per device: the current device must be the one the simulator's planes live on
  int dev = -1;
  CF_CUDA(cudaGetDevice(&dev));
  cudaPointerAttributes attr;
  CF_CUDA(cudaPointerGetAttributes(&attr, sim->state));
  if (attr.type != cudaMemoryTypeDevice && attr.type != cudaMemoryTypeManaged)
    return fail(CF_E_ARG, "cf_mppi_update_static: the simulator's workspace is not device memory");
  if (attr.type == cudaMemoryTypeDevice && attr.device != dev)
    return fail(CF_E_ARG, "cf_mppi_update_static: the simulator's workspace is on device %d but device %d is current",
                attr.device, dev);
  void *scratch = nullptr;
  rc = static_scratch_addr(dev, &scratch);
  if (rc != CF_OK) return rc;
  // from here on this is cf_mppi_update on that memory: it zeroes the completion counter on the stream (the rest of the
  // scratch is written before it is read, so the previous call's leftovers do no harm) and launches the same kernel
  return cf_mppi_update(sim, mp, nominal_dev, plan_dev, info_dev, elite_idx_dev, scratch, CF_MPPI_STATIC_SCRATCH_BYTES);
}

extern "C" int cf_mppi_iterate(cf_sim *sim, const cf_mppi_params *mp, const float *x0_dev, void *nominal_dev,
                               void *plan_dev, void *info_dev, int32_t *elite_idx_dev, void *scratch_dev,
                               size_t scratch_bytes) {
  int rc = check(sim, mp);
  if (rc != CF_OK) return rc;
  rc = cf_set_state(sim, x0_dev, 1);
  if (rc != CF_OK) return rc;
  rc = cf_step(sim, nominal_dev, mp->horizon, mp->cmd_hold, mp->horizon * mp->cmd_hold, 0, nullptr, 0);
  if (rc != CF_OK) return rc;
  return cf_mppi_update(sim, mp, nominal_dev, plan_dev, info_dev, elite_idx_dev, scratch_dev, scratch_bytes);
}

extern "C" int cf_mppi_iterate_host(cf_sim *sim, const cf_mppi_params *mp, const float *x0_host, void *nominal_dev,
                                    void *plan_host, void *info_host, void *plan_dev, void *info_dev,
                                    void *scratch_dev, size_t scratch_bytes) {
  int rc = check(sim, mp);
  if (rc != CF_OK) return rc;
  if (!x0_host || !plan_host || !info_host || !plan_dev || !info_dev) return fail(CF_E_ARG, "NULL argument");
  // the broadcast start state is parked in the workspace and consumed by the rollout launch (lazy cf_set_state)
  if (!sim->have_state) return fail(CF_E_STATE, "cf_mppi_iterate_host needs a prior cf_reset (world parameters)");
  CF_CUDA(cudaMemcpyAsync(sim->bcast_buf, x0_host, sizeof(float) * sim->D, cudaMemcpyHostToDevice, sim->stream));
  sim->pending_bcast = true; sim->rearmed = true; sim->md_valid = false; sim->cost_valid = false;   // = cf_set_state(broadcast)
  rc = cf_step(sim, nominal_dev, mp->horizon, mp->cmd_hold, mp->horizon * mp->cmd_hold, 0, nullptr, 0);
  if (rc != CF_OK) return rc;
  rc = cf_mppi_update(sim, mp, nominal_dev, plan_dev, info_dev, nullptr, scratch_dev, scratch_bytes);
  if (rc != CF_OK) return rc;
  CF_CUDA(cudaMemcpyAsync(plan_host, plan_dev, sizeof(float4) * mp->horizon, cudaMemcpyDeviceToHost, sim->stream));
  CF_CUDA(cudaMemcpyAsync(info_host, info_dev, sizeof(float) * CF_MPPI_INFO_WORDS(sim->p.n_ctrl), cudaMemcpyDeviceToHost,
                          sim->stream));
  CF_CUDA(cudaStreamSynchronize(sim->stream));
  return CF_OK;
}

extern "C" int cf_mppi_pack_best(cf_sim *sim, const cf_mppi_params *mp, const void *info_dev, const void *plan_dev,
                                 int ctrl_offset, float *row_dev) {
  int rc = check(sim, mp);
  if (rc != CF_OK) return rc;
  if (!info_dev || !plan_dev || !row_dev || ctrl_offset < 0) return fail(CF_E_ARG, "bad argument");
  pack_best_kernel<<<1, 128, 0, sim->stream>>>((const float *)info_dev, (const float4 *)plan_dev, sim->p.n_ctrl, mp->horizon,
                                               ctrl_offset, row_dev);
  CF_CUDA(cudaGetLastError());
  return CF_OK;
}

extern "C" int cf_mppi_select(cf_sim *sim, const float *rows_dev, int n_rows, int horizon, float *best_row_dev) {
  if (!sim || !rows_dev || !best_row_dev) return fail(CF_E_ARG, "NULL argument");
  if (n_rows < 1 || horizon < 1) return fail(CF_E_ARG, "n_rows, horizon >= 1");
  select_row_kernel<<<1, 128, 0, sim->stream>>>(rows_dev, n_rows, horizon, best_row_dev);
  CF_CUDA(cudaGetLastError());
  return CF_OK;
}
