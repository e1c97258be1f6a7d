// cf_depth.cu -- batched depth ray casting ("parallel rendering of depth images ... 64x64 ray resolution
// across 1,024 environments"; L286-L288).  Reading R34: pinhole camera rigidly attached to every drone,
// optical axis = body +x, static scene of spheres, axis-aligned boxes and the ground plane z = 0, depth = distance along
// the unit ray to the nearest surface, -1 for no hit within t_max.  Arithmetic, not graphics: no GL / Vulkan anywhere.
//
// thread = ray, block = one 16 x 16 pixel tile of ONE drone's image.  The block's first threads turn the drone's pose (read
// from the simulator's state planes) into camera origin + rotation, bound the tile's rays by a cone (axis = the tile
// centre's ray, half-angle = the widest corner) and CULL the scene against it: warp 0 tests the spheres, warp 2 the
// bounding spheres of the boxes (point-to-cone distance perp cos(a) - along sin(a) <= r, conservative: never drops a
// primitive a ray of the tile can hit), and ballot-compacts the survivors into shared memory as origin-relative
// constants.  A ray then intersects only the tile's few survivors (~11 instructions per sphere, ~20 per box, MUFU
// square root, branch-free slab test) and the image leaves as streaming stores.  Measured on the 33-primitive scene:
// 224 us (256 consecutive pixels per block, no culling, IEEE sqrt) -> 146 us (whole image per block) -> tile culling.
#include "cf_internal.h"

#include <cmath>
#include <cstring>

using namespace cf;

namespace {

constexpr int kTile = 16;           // 16 x 16 pixel tiles, one block of 256 threads each
constexpr int kBlock = kTile * kTile;

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
  __shared__ float sR[9], so[3], s_cone[5];               // rotation, origin, tile cone: axis (world), cos, sin of the half-angle
  __shared__ float4 s_sph[CF_DEPTH_MAX_PRIMS];            // surviving spheres: (c - o, r^2)
  __shared__ float4 s_lo[CF_DEPTH_MAX_PRIMS], s_hi[CF_DEPTH_MAX_PRIMS];        // surviving box slabs relative to the origin
  __shared__ int s_n[2];
  const long long i = blockIdx.x;                         // drone
  const int tid = threadIdx.x, lane = tid & 31;
  const int tiles_x = (A.W + kTile - 1) / kTile;
  const int ty0 = (blockIdx.y / tiles_x) * kTile, tx0 = (blockIdx.y % tiles_x) * kTile;
  const int tx1 = min(tx0 + kTile, A.W), ty1 = min(ty0 + kTile, A.H);          // the tile covers pixels [tx0, tx1) x [ty0, ty1)
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
    // bounding cone of the tile in the body frame: the tile is the rectangle [y0, y1] x [z0, z1] on the plane x = 1
    const float y0 = -((float)tx0 - 0.5f * (float)A.W) * A.pix, y1 = -((float)tx1 - 0.5f * (float)A.W) * A.pix;
    const float z0 = -((float)ty0 - 0.5f * (float)A.H) * A.pix, z1 = -((float)ty1 - 0.5f * (float)A.H) * A.pix;
    const float yc = 0.5f * (y0 + y1), zc = 0.5f * (z0 + z1);
    const float ic = rsqrtf(1.0f + yc * yc + zc * zc);
    float cmin = 1.0f;                                    // cos of the widest corner angle
    const float ys[2] = { y0, y1 }, zs[2] = { z0, z1 };
#pragma unroll
    for (int a = 0; a < 2; ++a)
#pragma unroll
      for (int b = 0; b < 2; ++b)
        cmin = fminf(cmin, (1.0f + ys[a] * yc + zs[b] * zc) * ic * rsqrtf(1.0f + ys[a] * ys[a] + zs[b] * zs[b]));
    cmin = fmaxf(cmin - 1e-5f, 0.0f);                     // margin for the float32 arithmetic above (conservative)
#pragma unroll
    for (int r = 0; r < 3; ++r) s_cone[r] = (R[r][0] + R[r][1] * yc + R[r][2] * zc) * ic;
    s_cone[3] = cmin;
    s_cone[4] = sqrtf(fmaxf(1.0f - cmin * cmin, 0.0f));
  }
  __syncthreads();
  // cull: a sphere (centre m relative to the origin, radius r) can be hit by a ray inside the cone only if its centre is
  // within r of the cone: perp cos(a) - along sin(a) <= r (<= |m|, so a sphere containing the origin always passes)
  auto near_cone = [&](float mx, float my, float mz, float r) {
    const float along = mx * s_cone[0] + my * s_cone[1] + mz * s_cone[2];
    const float m2 = mx * mx + my * my + mz * mz;
    const float perp = sqrtf(fmaxf(m2 - along * along, 0.0f));
    return perp * s_cone[3] - along * s_cone[4] <= r + 1e-4f * (1.0f + sqrtf(m2));
  };
  if (tid < 32) {
    const bool have = tid < A.n_spheres;
    const float mx = have ? A.spheres[tid][0] - so[0] : 0.f, my = have ? A.spheres[tid][1] - so[1] : 0.f;
    const float mz = have ? A.spheres[tid][2] - so[2] : 0.f, r = have ? A.spheres[tid][3] : 0.f;
    const bool vis = have && near_cone(mx, my, mz, r);
    const unsigned mask = __ballot_sync(0xffffffffu, vis);
    if (vis) s_sph[__popc(mask & ((1u << lane) - 1u))] = make_float4(mx, my, mz, r * r);
    if (lane == 0) s_n[0] = __popc(mask);
  } else if (tid >= 64 && tid < 96) {
    const int b = tid - 64;
    const bool have = b < A.n_boxes;
    float c[3] = { 0, 0, 0 }, hf[3] = { 0, 0, 0 };
    if (have) {
#pragma unroll
      for (int j = 0; j < 3; ++j) { c[j] = A.boxes[b][j] - so[j]; hf[j] = A.boxes[b][3 + j]; }
    }
    const bool vis = have && near_cone(c[0], c[1], c[2], sqrtf(hf[0] * hf[0] + hf[1] * hf[1] + hf[2] * hf[2]));
    const unsigned mask = __ballot_sync(0xffffffffu, vis);
    if (vis) {
      const int pos = __popc(mask & ((1u << lane) - 1u));
      s_lo[pos] = make_float4(c[0] - hf[0], c[1] - hf[1], c[2] - hf[2], 0.f);
      s_hi[pos] = make_float4(c[0] + hf[0], c[1] + hf[1], c[2] + hf[2], 0.f);
    }
    if (lane == 0) s_n[1] = __popc(mask);
  }
  __syncthreads();
  const int u = tx0 + (tid & (kTile - 1)), v = ty0 + tid / kTile;
  if (u >= A.W || v >= A.H) return;
  const int n_sph = s_n[0], n_box = s_n[1];
  const float INF = __int_as_float(0x7f800000);
  {
    // d_body = normalise(1, -(u + 1/2 - W/2) s, -(v + 1/2 - H/2) s);  d = R d_body
    const float by = -((float)u + 0.5f - 0.5f * (float)A.W) * A.pix, bz = -((float)v + 0.5f - 0.5f * (float)A.H) * A.pix;
    const float inv = rsqrtf(1.0f + by * by + bz * bz);
    const float dx = (sR[0] + sR[1] * by + sR[2] * bz) * inv;
    const float dy = (sR[3] + sR[4] * by + sR[5] * bz) * inv;
    const float dz = (sR[6] + sR[7] * by + sR[8] * bz) * inv;
    float best = INF;
    // spheres: with m = c - o, b = m.d, perpendicular part l = m - b d: disc = r^2 - |l|^2, t = b -+ sqrt(disc)
    for (int s = 0; s < n_sph; ++s) {
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
    if (n_box > 0) {
      const float ix = dx != 0.0f ? 1.0f / dx : 1e30f, iy = dy != 0.0f ? 1.0f / dy : 1e30f, iz = dz != 0.0f ? 1.0f / dz : 1e30f;
      for (int b = 0; b < n_box; ++b) {
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
    __stcs(A.depth + (size_t)i * A.W * A.H + (size_t)v * A.W + u, (best <= A.t_max && best < INF) ? best : -1.0f);
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
  const int chunks = ((dp->width + kTile - 1) / kTile) * ((dp->height + kTile - 1) / kTile);
  if (chunks > 65535) return fail(CF_E_ARG, "image too large");
  dim3 grid((unsigned)sim->MN, (unsigned)chunks);
  depth_kernel<<<grid, kBlock, 0, sim->stream>>>(A);
  CF_CUDA(cudaGetLastError());
  return CF_OK;
}

// The same rendering driven from HOST buffers (the end-to-end path): state_host [D][MN] (the poses; NULL = render the
// simulator's current state) is copied host->device into the state planes, the images are rendered into staging_dev and
// copied device->host, and the stream is synchronised.
extern "C" int cf_depth_host(cf_sim *sim, const cf_depth_params *dp, const float *state_host, float *depth_host,
                             float *staging_dev, size_t staging_bytes) {
  if (!sim || !dp || !depth_host || !staging_dev) return fail(CF_E_ARG, "NULL argument");
  if (dp->struct_size != sizeof(cf_depth_params)) return fail(CF_E_ARG, "cf_depth_params.struct_size mismatch");
  if (dp->width < 1 || dp->height < 1) return fail(CF_E_ARG, "bad image size");
  const size_t bytes = sizeof(float) * (size_t)sim->MN * (size_t)dp->width * (size_t)dp->height;
  if (staging_bytes < bytes) return fail(CF_E_BUFFER, "staging too small: %zu < %zu", staging_bytes, bytes);
  if (state_host) {
    if (!sim->have_state) return fail(CF_E_STATE, "cf_depth_host needs a prior cf_reset (world parameters)");
    int rc = cf_materialise(sim);
    if (rc != CF_OK) return rc;
    CF_CUDA(cudaMemcpyAsync(sim->state, state_host, sizeof(float) * sim->D * (size_t)sim->MN, cudaMemcpyHostToDevice, sim->stream));
    sim->md_valid = false; sim->cost_valid = false; sim->rearmed = false;
  }
  int rc = cf_depth(sim, dp, staging_dev);
  if (rc != CF_OK) return rc;
  CF_CUDA(cudaMemcpyAsync(depth_host, staging_dev, bytes, cudaMemcpyDeviceToHost, sim->stream));
  CF_CUDA(cudaStreamSynchronize(sim->stream));
  return CF_OK;
}
