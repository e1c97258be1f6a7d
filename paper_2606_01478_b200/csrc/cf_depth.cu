// cf_depth.cu -- batched depth ray casting ("parallel rendering of depth images ... 64x64 ray resolution
// across 1,024 environments"; L286-L288).  Reading R34: pinhole camera rigidly attached to every drone,
// optical axis = body +x, static scene of spheres, axis-aligned boxes and the ground plane z = 0, depth = distance along
// the unit ray to the nearest surface, -1 for no hit within t_max.  Arithmetic, not graphics: no GL / Vulkan anywhere.
//
// thread = ray.  A block renders up to kRaysPerThread x 256 pixels of ONE drone: its first threads turn the drone's pose
// (read from the simulator's state planes) and the scene into per-drone constants in shared memory (camera origin,
// rotation, origin-relative sphere centres, origin-relative box slabs as float4), so a ray costs ~11 instructions per
// sphere and ~20 per box (MUFU square root, branch-free slab test); the image leaves as coalesced streaming stores.
// First version (256 pixels per block, IEEE sqrt, per-axis parallel-ray branches): 224 us per 1024 x 64 x 64 image batch.
#include "cf_internal.h"

#include <cmath>
#include <cstring>

using namespace cf;

namespace {

constexpr int kBlock = 256;
constexpr int kRaysPerThread = 16;     // a 64 x 64 image is one block: the per-drone setup is paid once

struct DepthArgs {
  const float *state;      // [D][MN]
  float *depth;            // [MN][H][W]
  long long MN;
  int model, W, H;
  float pix;               // 2 tan(fov_x / 2) / W
  float t_max;
  float cam_offset[3];
  int n_spheres, n_boxes, ground_plane;
  float spheres[CF_DEPTH_MAX_PRIMS][4];
  float boxes[CF_DEPTH_MAX_PRIMS][6];
};

__global__ void __launch_bounds__(kBlock)
depth_kernel(const __grid_constant__ DepthArgs A) {
  __shared__ float sR[9], so[3];
  __shared__ float4 s_sph[CF_DEPTH_MAX_PRIMS];            // (c - o, r^2)
  __shared__ float4 s_lo[CF_DEPTH_MAX_PRIMS], s_hi[CF_DEPTH_MAX_PRIMS];        // box slabs relative to the origin
  const long long i = blockIdx.x;                         // drone
  const int tid = threadIdx.x;
  if (tid == 0) {
    const long long MN = A.MN;
    float R[3][3];
    if (A.model == MODEL_FP) {
      float q[4] = { A.state[3 * MN + i], A.state[4 * MN + i], A.state[5 * MN + i], A.state[6 * MN + i] };
      quat_to_R(q, R);
    } else {
      euler_to_R(A.state[3 * MN + i], A.state[4 * MN + i], A.state[5 * MN + i], R);
    }
#pragma unroll
    for (int r = 0; r < 3; ++r) {
#pragma unroll
      for (int c = 0; c < 3; ++c) sR[3 * r + c] = R[r][c];
      so[r] = A.state[r * MN + i] + R[r][0] * A.cam_offset[0] + R[r][1] * A.cam_offset[1] + R[r][2] * A.cam_offset[2];
    }
  }
  __syncthreads();
  if (tid < A.n_spheres) {
    s_sph[tid] = make_float4(A.spheres[tid][0] - so[0], A.spheres[tid][1] - so[1], A.spheres[tid][2] - so[2],
                             A.spheres[tid][3] * A.spheres[tid][3]);
  } else if (tid >= 64 && tid - 64 < A.n_boxes) {
    const int b = tid - 64;
    float lo[3], hi[3];
#pragma unroll
    for (int j = 0; j < 3; ++j) {
      lo[j] = (A.boxes[b][j] - A.boxes[b][3 + j]) - so[j];
      hi[j] = (A.boxes[b][j] + A.boxes[b][3 + j]) - so[j];
    }
    s_lo[b] = make_float4(lo[0], lo[1], lo[2], 0.f);
    s_hi[b] = make_float4(hi[0], hi[1], hi[2], 0.f);
  }
  __syncthreads();
  const int HW = A.W * A.H;
  const float INF = __int_as_float(0x7f800000);
  const int pix_end = min(HW, (int)(blockIdx.y + 1) * kBlock * kRaysPerThread);
  for (int pix = blockIdx.y * kBlock * kRaysPerThread + tid; pix < pix_end; pix += kBlock) {
    const int v = pix / A.W, u = pix - v * A.W;
    // d_body = normalise(1, -(u + 1/2 - W/2) s, -(v + 1/2 - H/2) s);  d = R d_body
    const float by = -((float)u + 0.5f - 0.5f * (float)A.W) * A.pix, bz = -((float)v + 0.5f - 0.5f * (float)A.H) * A.pix;
    const float inv = rsqrtf(1.0f + by * by + bz * bz);
    const float dx = (sR[0] + sR[1] * by + sR[2] * bz) * inv;
    const float dy = (sR[3] + sR[4] * by + sR[5] * bz) * inv;
    const float dz = (sR[6] + sR[7] * by + sR[8] * bz) * inv;
    float best = INF;
    // spheres: with m = c - o, b = m.d, perpendicular part l = m - b d: disc = r^2 - |l|^2, t = b -+ sqrt(disc)
    for (int s = 0; s < A.n_spheres; ++s) {
      const float4 m = s_sph[s];
      const float b = m.x * dx + m.y * dy + m.z * dz;
      const float lx = m.x - b * dx, ly = m.y - b * dy, lz = m.z - b * dz;
      const float disc = m.w - (lx * lx + ly * ly + lz * lz);
      const float sq = mufu_sqrt(fmaxf(disc, 0.0f));
      const float t0 = b - sq, t1 = b + sq;
      const float t = t0 > 0.0f ? t0 : t1;
      best = fminf(best, (disc >= 0.0f && t > 0.0f) ? t : INF);
    }
    // boxes: slab method.  A ray parallel to a slab (d_j == 0) is inside it iff lo_j <= 0 <= hi_j; taking 1/d_j = 1e30
    // there reproduces exactly that rule without a branch per box (lo 1e30, hi 1e30 are -huge / +huge inside the slab,
    // same-signed outside, and 0 * 1e30 = 0 on a face: no 0 * inf)
    if (A.n_boxes > 0) {
      const float ix = dx != 0.0f ? 1.0f / dx : 1e30f, iy = dy != 0.0f ? 1.0f / dy : 1e30f, iz = dz != 0.0f ? 1.0f / dz : 1e30f;
      for (int b = 0; b < A.n_boxes; ++b) {
        const float4 lo = s_lo[b], hi = s_hi[b];
        const float ax = lo.x * ix, bx = hi.x * ix, ay = lo.y * iy, by2 = hi.y * iy, az = lo.z * iz, bz2 = hi.z * iz;
        const float t_in = fmaxf(fmaxf(fminf(ax, bx), fminf(ay, by2)), fminf(az, bz2));
        const float t_out = fminf(fminf(fmaxf(ax, bx), fmaxf(ay, by2)), fmaxf(az, bz2));
        const float t = t_in > 0.0f ? t_in : t_out;
        best = fminf(best, (t_in <= t_out && t > 0.0f) ? t : INF);
      }
    }
    if (A.ground_plane && dz != 0.0f) {
      const float t = -so[2] / dz;
      if (t > 0.0f) best = fminf(best, t);
    }
    __stcs(A.depth + (size_t)i * HW + pix, (best <= A.t_max && best < INF) ? best : -1.0f);
  }
}

}  // namespace

extern "C" int cf_depth(cf_sim *sim, const cf_depth_params *dp, float *depth_dev) {
  if (!sim || !dp || !depth_dev) return fail(CF_E_ARG, "NULL argument");
  if (dp->struct_size != sizeof(cf_depth_params)) return fail(CF_E_ARG, "cf_depth_params.struct_size mismatch");
  if (dp->width < 1 || dp->height < 1 || (long long)dp->width * dp->height > (1 << 24)) return fail(CF_E_ARG, "bad image size");
  if (!(dp->fov_x > 0.f && dp->fov_x < 3.1f)) return fail(CF_E_ARG, "fov_x must be in (0, 3.1) rad");
  if (dp->n_spheres < 0 || dp->n_spheres > CF_DEPTH_MAX_PRIMS || dp->n_boxes < 0 || dp->n_boxes > CF_DEPTH_MAX_PRIMS)
    return fail(CF_E_ARG, "at most %d spheres and %d boxes", CF_DEPTH_MAX_PRIMS, CF_DEPTH_MAX_PRIMS);
  if (!sim->have_state) return fail(CF_E_STATE, "cf_depth before cf_reset");
  int rc = cf_materialise(sim);
  if (rc != CF_OK) return rc;
  DepthArgs A;
  A.state = sim->state; A.depth = depth_dev; A.MN = sim->MN; A.model = sim->model; A.W = dp->width; A.H = dp->height;
  A.pix = (float)(2.0 * std::tan(0.5 * (double)dp->fov_x) / dp->width);
  A.t_max = dp->t_max > 0.f ? dp->t_max : INFINITY;
  for (int j = 0; j < 3; ++j) A.cam_offset[j] = dp->cam_offset[j];
  A.n_spheres = dp->n_spheres; A.n_boxes = dp->n_boxes; A.ground_plane = dp->ground_plane;
  memcpy(A.spheres, dp->spheres, sizeof(A.spheres));
  memcpy(A.boxes, dp->boxes, sizeof(A.boxes));
  const int per_block = kBlock * kRaysPerThread;
  const int chunks = (dp->width * dp->height + per_block - 1) / per_block;
  if (chunks > 65535) return fail(CF_E_ARG, "image too large");
  dim3 grid((unsigned)sim->MN, (unsigned)chunks);
  depth_kernel<<<grid, kBlock, 0, sim->stream>>>(A);
  CF_CUDA(cudaGetLastError());
  return CF_OK;
}
