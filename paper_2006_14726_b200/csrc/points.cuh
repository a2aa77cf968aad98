// points.cuh -- the comparison renderer of the paper: the 2.5D point
// rendering of [ZAL12], "the authors render the image pixels as point primitives on the GPU"
// (PAPER.md:37), object-space coordinate -> "window coordinates by applying the viewing and camera
// transforms as well as viewport transform", point size "fixed to a certain number
// of pixels", depth test per point, not per fragment.  The paper
// runs it through OpenGL (unavailable on this box); this is the same rasterisation as three CUDA
// kernels over the splats of the latest update: depth (64-bit atomicMin on (view depth, splat
// id)), colour (the winner of a pixel writes its stored colour), background (+ re-arming the
// depth buffer for the next call).
#pragma once
#include "common.cuh"

namespace sw {

constexpr int POINT_THREADS = 256;
constexpr uint64_t ZKEY_EMPTY = ~0ull;

struct PointParams {
  DevCamera cam;
  const float4* sphere;   // sorted order: centre xyz (radius unused)
  const float4* rgba;
  const uint32_t* ids;
  const FrameState* st;
  uint64_t* zkey;         // one per destination pixel, ZKEY_EMPTY between calls
  float4* out;
  int point_px;
  float hW, hH, off;      // W2 / 2, H2 / 2, point_px / 2 + 1/2 (all exact)
};

// Window position of splat i: false if it is culled.  zc = view-axis depth (> 0), (x0, y0) = the
// first pixel of its point_px x point_px square (w - size/2 < pixel centre <= w + size/2).
__device__ __forceinline__ bool project_point(const PointParams& p, const float4 c, float& zc, int& x0, int& y0) {
  const DevCamera& cam = p.cam;
  const float vx = sub_(c.x, cam.e[0]), vy = sub_(c.y, cam.e[1]), vz = sub_(c.z, cam.e[2]);
  zc = fma_(vz, cam.F[2], fma_(vy, cam.F[1], mul_(vx, cam.F[0])));
  if (!(zc > 0.0f)) return false;
  const float xr = fma_(vz, cam.R[2], fma_(vy, cam.R[1], mul_(vx, cam.R[0])));
  const float yu = fma_(vz, cam.U[2], fma_(vy, cam.U[1], mul_(vx, cam.U[0])));
  const float ndx = div_(xr, mul_(zc, cam.ta)), ndy = div_(yu, mul_(zc, cam.tau));
  const float wx = fma_(ndx, p.hW, p.hW), wy = fma_(-ndy, p.hH, p.hH);
  const float fx0 = add_(floorf(sub_(wx, p.off)), 1.0f), fy0 = add_(floorf(sub_(wy, p.off)), 1.0f);
  if (!(fx0 > -1e9f && fx0 < 1e9f && fy0 > -1e9f && fy0 < 1e9f)) return false;
  x0 = (int)fx0;
  y0 = (int)fy0;
  return true;
}

template <bool COLOUR>
__global__ void __launch_bounds__(POINT_THREADS)
points_kernel(const PointParams p) {
  const int n = (int)p.st->n;
  const int W = p.cam.W, H = p.cam.H;
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
    float zc;
    int x0, y0;
    if (!project_point(p, __ldg(p.sphere + i), zc, x0, y0)) continue;
    if (x0 >= W || y0 >= H || x0 + p.point_px <= 0 || y0 + p.point_px <= 0) continue;
    const uint64_t key = ((uint64_t)__float_as_uint(zc) << 32) | __ldg(p.ids + i);   // zc > 0: bits are ordered
    float4 col;
    if (COLOUR) col = __ldg(p.rgba + i);
    for (int y = max(y0, 0); y < min(y0 + p.point_px, H); ++y)
      for (int x = max(x0, 0); x < min(x0 + p.point_px, W); ++x) {
        const size_t px = (size_t)y * W + x;
        if (COLOUR) {
          if (p.zkey[px] == key) p.out[px] = col;
        } else {
          atomicMin(reinterpret_cast<unsigned long long*>(p.zkey + px), (unsigned long long)key);
        }
      }
  }
}

// Pixels no point covers are background (0,0,0,0); every depth entry goes back to "empty".
__global__ void __launch_bounds__(POINT_THREADS)
points_background_kernel(const PointParams p) {
  const int64_t total = (int64_t)p.cam.W * p.cam.H;
  for (int64_t px = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; px < total; px += (int64_t)gridDim.x * blockDim.x) {
    if (p.zkey[px] == ZKEY_EMPTY) p.out[px] = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
    else p.zkey[px] = ZKEY_EMPTY;
  }
}

}  // namespace sw
