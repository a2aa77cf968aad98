// march.cuh -- the server's volume ray marcher (first half).
// PAPER.md:63 sec. 4.1: "we render the volume using a ray marcher that employs one of the
// heuristics presented by Zellmann et al. to estimate which depth value represents the volume
// best.  We march rays r = o + d t"; sec. 4.2: it "writes out colors and t values to
// an off-screen buffer".  Recipe = BASELINE.json's server pass (S12): unit cube, n^3
// float32 densities at voxel centres, manual trilinear interpolation (texture units filter with
// 9-bit weights and would not be bit-identical to the oracle), opacity tents, premultiplied
// front-to-back compositing, depth = t of the first sample whose accumulated alpha reaches
// depth_alpha, early termination at stop_alpha.
//
// One thread per pixel, one warp per 8x4 pixel tile: the 32 rays of a warp sample neighbouring
// voxels, so the eight loads per sample hit the same few L1 lines; the volumes of the
// configs (<= 512 MB) are L2 resident only up to 256^3, the rest streams from HBM once per frame.
#pragma once
#include "common.cuh"

namespace sw {

constexpr int MARCH_THREADS = 128;

struct MarchParams {
  const float* __restrict__ vol;
  int n;
  float fn, step;   // float(n), 0.5 / n
  int n_tents;
  float iso[4], amax[4], rgb[4][3];
  float hw, shade, one_minus_shade, depth_alpha, stop_alpha;
  DevCamera cam;
  float4* __restrict__ color;
  float* __restrict__ depth;
};

__device__ __forceinline__ float lerp_(float a, float b, float f) { return fma_(f, sub_(b, a), a); }

__global__ void __launch_bounds__(MARCH_THREADS)
march_kernel(const MarchParams p) {
  const DevCamera& cam = p.cam;
  const int tiles_x = (cam.W + 7) >> 3, tiles_y = (cam.H + 3) >> 2;
  const int lane = threadIdx.x & 31;
  const int n = p.n;
  const float INF = __int_as_float(0x7f800000);
  for (int tile = blockIdx.x * (MARCH_THREADS / 32) + (threadIdx.x >> 5); tile < tiles_x * tiles_y;
       tile += gridDim.x * (MARCH_THREADS / 32)) {
    const int ty = tile / tiles_x, tx = tile - ty * tiles_x;
    const int x = tx * 8 + (lane & 7), y = ty * 4 + (lane >> 3);
    if (x >= cam.W || y >= cam.H) continue;
    float d[3], len;
    pixel_ray(cam, x, y, d, len);
    float t0 = 0.0f, t1 = INF;
    bool miss = false;
#pragma unroll
    for (int k = 0; k < 3; ++k) {
      if (fabsf(d[k]) < 1e-30f) {
        if (cam.e[k] < 0.0f || cam.e[k] > 1.0f) miss = true;
      } else {
        float a = div_(sub_(0.0f, cam.e[k]), d[k]), b = div_(sub_(1.0f, cam.e[k]), d[k]);
        if (a > b) { const float s = a; a = b; b = s; }
        t0 = fmaxf(t0, a);
        t1 = fminf(t1, b);
      }
    }
    float C[3] = {0.0f, 0.0f, 0.0f}, A = 0.0f, tdepth = 0.0f;
    if (!miss && t0 < t1) {
      for (int s = 0;; ++s) {
        const float t = fma_(add_(__int2float_rn(s), 0.5f), p.step, t0);
        if (!(t < t1)) break;
        float P[3], f[3];
        int i0[3], i1[3];
#pragma unroll
        for (int k = 0; k < 3; ++k) {
          P[k] = fma_(t, d[k], cam.e[k]);
          const float g = fma_(P[k], p.fn, -0.5f);
          const float fl = floorf(g);
          f[k] = sub_(g, fl);
          const int a = (int)fl;
          i0[k] = min(max(a, 0), n - 1);
          i1[k] = min(max(a + 1, 0), n - 1);
        }
        const size_t r00 = ((size_t)i0[2] * n + i0[1]) * n, r10 = ((size_t)i0[2] * n + i1[1]) * n;
        const size_t r01 = ((size_t)i1[2] * n + i0[1]) * n, r11 = ((size_t)i1[2] * n + i1[1]) * n;
        const float v000 = __ldg(p.vol + r00 + i0[0]), v100 = __ldg(p.vol + r00 + i1[0]);
        const float v010 = __ldg(p.vol + r10 + i0[0]), v110 = __ldg(p.vol + r10 + i1[0]);
        const float v001 = __ldg(p.vol + r01 + i0[0]), v101 = __ldg(p.vol + r01 + i1[0]);
        const float v011 = __ldg(p.vol + r11 + i0[0]), v111 = __ldg(p.vol + r11 + i1[0]);
        const float c00 = lerp_(v000, v100, f[0]), c10 = lerp_(v010, v110, f[0]);
        const float c01 = lerp_(v001, v101, f[0]), c11 = lerp_(v011, v111, f[0]);
        const float dens = lerp_(lerp_(c00, c10, f[1]), lerp_(c01, c11, f[1]), f[2]);
        float alpha = 0.0f;
        int ci = -1;
#pragma unroll
        for (int i = 0; i < 4; ++i) {
          if (i < p.n_tents) {
            const float w = sub_(1.0f, div_(fabsf(sub_(dens, p.iso[i])), p.hw));
            if (w > 0.0f) {
              alpha = fma_(p.amax[i], w, alpha);
              if (ci < 0) ci = i;
            }
          }
        }
        if (alpha > 0.0f) {
          const float T = sub_(1.0f, A), Ta = mul_(T, alpha);
#pragma unroll
          for (int k = 0; k < 3; ++k) {
            const float pc = fminf(fmaxf(P[k], 0.0f), 1.0f);
            const float mod = fma_(p.shade, pc, p.one_minus_shade);
            // constant-index selects instead of a dynamically indexed parameter array
            const float base = ci == 0 ? p.rgb[0][k] : ci == 1 ? p.rgb[1][k] : ci == 2 ? p.rgb[2][k] : p.rgb[3][k];
            C[k] = fma_(Ta, mul_(base, mod), C[k]);
          }
          A = fma_(T, alpha, A);
          if (tdepth == 0.0f && A >= p.depth_alpha) tdepth = t;
          if (A >= p.stop_alpha) break;
        }
      }
    }
    const size_t px = (size_t)y * cam.W + x;
    p.color[px] = make_float4(C[0], C[1], C[2], A);
    p.depth[px] = tdepth;
  }
}

}  // namespace sw
