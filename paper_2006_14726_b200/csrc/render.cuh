// render.cuh -- step a6 of SURVEY.md sec. 8(a): per-pixel software BVH traversal of the sphere
// splats with front-to-back compositing of every entry hit ("render them as a point cloud
// using ray tracing"; "spheres that are represented as real quadrics",
// PAPER.md:55; CUDA software ray tracing without RT cores).
//
// One thread per destination pixel, one warp per 8x4 pixel tile, four warps (16x8 pixels)
// per block.  Traversal keeps the K nearest hits beyond a cursor (t, id) in a register
// k-buffer sorted by (t, id); after the walk they are composited in order, and if the ray is
// not yet opaque (alpha < 0.99) and the k-buffer was full (hits may have been dropped), the ray is
// re-launched from the last composited (t, id).  The result is exactly "sort all hits by
// (t, id), composite until alpha >= 0.99" (oracle step O9), whatever K is.
//
// The traversal stack lives in shared memory ([depth][thread], conflict free) with a
// local-memory tail so that any legal tree depth (<= 63 key bits + 32 index bits) works.
#pragma once
#include "common.cuh"

namespace sw {

constexpr int RENDER_THREADS = 128;
constexpr int KBUF = 8;
constexpr int SSTACK = 24;
constexpr int LSTACK = 72;
constexpr uint32_t EMPTY_LEAF = 0xffffffffu;

struct RenderParams {
  DevCamera cam;
  const Node* nodes;
  const float4* sphere;
  const float4* rgba;
  const uint32_t* ids;
  const FrameState* st;
  float4* out;
};

#ifdef SPLATS_STATS
// Debug build only (-DSPLATS_STATS): traversal counters, read back with splats_debug_stats().
__device__ unsigned long long g_stats[8];  // 0 node visits, 1 leaf tests, 2 hits kept, 3 passes, 4 rays past root, 5 max stack
#define STAT_ADD(i, v) atomicAdd(&g_stats[i], (unsigned long long)(v))
#define STAT_MAX(i, v) atomicMax(&g_stats[i], (unsigned long long)(v))
#else
#define STAT_ADD(i, v)
#define STAT_MAX(i, v)
#endif

struct KBuffer {
  float t[KBUF];
  uint32_t leaf[KBUF];
  __device__ __forceinline__ void clear() {
#pragma unroll
    for (int i = 0; i < KBUF; ++i) { t[i] = __int_as_float(0x7f800000); leaf[i] = EMPTY_LEAF; }
  }
  // A full buffer may have dropped hits (evicted here, or culled by the t <= t[K-1] bound).
  __device__ __forceinline__ bool full() const { return leaf[KBUF - 1] != EMPTY_LEAF; }
  // sorted insertion by (t, id); the largest entry falls out when the buffer is full
  __device__ __forceinline__ void insert(float ct, uint32_t cl, const uint32_t* __restrict__ ids) {
#pragma unroll
    for (int i = 0; i < KBUF; ++i) {
      bool lt = ct < t[i];
      if (!lt && ct == t[i] && leaf[i] != EMPTY_LEAF && cl != EMPTY_LEAF) lt = __ldg(ids + cl) < __ldg(ids + leaf[i]);
      if (lt) {
        const float tt = t[i]; t[i] = ct; ct = tt;
        const uint32_t tl = leaf[i]; leaf[i] = cl; cl = tl;
      }
    }
  }
};

// Oracle step O8: entry t of the unit-direction ray (o, d) with sphere s; perpendicular-vector
// form of the discriminant (robust for small, distant spheres).
__device__ __forceinline__ bool ray_sphere(const float o[3], const float d[3], const float4 s, float& t) {
  const float ocx = sub_(s.x, o[0]), ocy = sub_(s.y, o[1]), ocz = sub_(s.z, o[2]);
  const float b = fma_(ocz, d[2], fma_(ocy, d[1], mul_(ocx, d[0])));
  const float lx = fma_(-b, d[0], ocx), ly = fma_(-b, d[1], ocy), lz = fma_(-b, d[2], ocz);
  const float l2 = fma_(lz, lz, fma_(ly, ly, mul_(lx, lx)));
  const float disc = fma_(s.w, s.w, -l2);
  if (!(disc > 0.0f)) return false;
  t = sub_(b, sqrt_(disc));
  return t >= 0.0f;
}

__global__ void __launch_bounds__(RENDER_THREADS)
render_kernel(RenderParams prm) {
  __shared__ int s_stack[SSTACK][RENDER_THREADS];
  int l_stack[LSTACK];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const DevCamera& cam = prm.cam;
  const int x = blockIdx.x * 16 + (warp & 1) * 8 + (lane & 7);
  const int y = blockIdx.y * 8 + (warp >> 1) * 4 + (lane >> 3);
  const bool inside = x < cam.W && y < cam.H;
  const int n = (int)prm.st->n;

  float o[3] = {cam.e[0], cam.e[1], cam.e[2]};
  float d[3], len;
  pixel_ray(cam, min(x, cam.W - 1), min(y, cam.H - 1), d, len);

  // conservative slab test: boxes padded by far more than the float32 error of ray_sphere()
  float m = 1.0f;
#pragma unroll
  for (int a = 0; a < 3; ++a)
    m = fmaxf(m, fmaxf(fabsf(o[a]), fmaxf(fabsf(prm.st->root_lo[a]), fabsf(prm.st->root_hi[a]))));
  const float pad = 4e-5f * m;
  float idir[3], op[3], om[3];
#pragma unroll
  for (int a = 0; a < 3; ++a) { idir[a] = 1.0f / d[a]; op[a] = o[a] + pad; om[a] = o[a] - pad; }

  float C[3] = {0.0f, 0.0f, 0.0f}, A = 0.0f;
  float cur_t = -1.0f;
  uint32_t cur_id = 0;
  bool finished = !inside || n == 0;
  KBuffer kb;

  while (__any_sync(0xffffffffu, !finished)) {
    if (!finished) {
      kb.clear();
      const float t_lo = fmaxf(cur_t, 0.0f);
      STAT_ADD(3, 1);

      auto test_leaf = [&](uint32_t leaf) {
        const float4 s = __ldg(prm.sphere + leaf);
        float t;
        STAT_ADD(1, 1);
        if (ray_sphere(o, d, s, t)) {
          if (t > cur_t || (t == cur_t && __ldg(prm.ids + leaf) > cur_id)) kb.insert(t, leaf, prm.ids);
        }
      };

      if (n == 1) {
        test_leaf(0u);
      } else {
        int sp = 0, node = 0;
        while (true) {
          const float4* np = reinterpret_cast<const float4*>(prm.nodes + node);
          const float4 n0 = __ldg(np), n1 = __ldg(np + 1), n2 = __ldg(np + 2), n3 = __ldg(np + 3);
          STAT_ADD(0, 1);
          STAT_MAX(5, sp);
          const float t_hi = kb.t[KBUF - 1];
          // left box: lo (n0.x n0.y n0.z) hi (n0.w n1.x n1.y); right box: lo (n1.z n1.w n2.x) hi (n2.y n2.z n2.w)
          float a0 = (n0.x - op[0]) * idir[0], a1 = (n0.w - om[0]) * idir[0];
          float b0 = (n0.y - op[1]) * idir[1], b1 = (n1.x - om[1]) * idir[1];
          float c0 = (n0.z - op[2]) * idir[2], c1 = (n1.y - om[2]) * idir[2];
          const float tnl = fmaxf(fmaxf(fminf(a0, a1), fminf(b0, b1)), fmaxf(fminf(c0, c1), t_lo));
          const float tfl = fminf(fminf(fmaxf(a0, a1), fmaxf(b0, b1)), fminf(fmaxf(c0, c1), t_hi));
          a0 = (n1.z - op[0]) * idir[0]; a1 = (n2.y - om[0]) * idir[0];
          b0 = (n1.w - op[1]) * idir[1]; b1 = (n2.z - om[1]) * idir[1];
          c0 = (n2.x - op[2]) * idir[2]; c1 = (n2.w - om[2]) * idir[2];
          const float tnr = fmaxf(fmaxf(fminf(a0, a1), fminf(b0, b1)), fmaxf(fminf(c0, c1), t_lo));
          const float tfr = fminf(fminf(fmaxf(a0, a1), fmaxf(b0, b1)), fminf(fmaxf(c0, c1), t_hi));
          bool hl = tnl <= tfl, hr = tnr <= tfr;
          const int cl = __float_as_int(n3.x), cr = __float_as_int(n3.y);
          if (hl && cl < 0) { test_leaf((uint32_t)~cl); hl = false; }
          if (hr && cr < 0) { test_leaf((uint32_t)~cr); hr = false; }
          if (hl && hr) {
            const bool left_first = tnl <= tnr;
            const int far = left_first ? cr : cl;
            node = left_first ? cl : cr;
            if (sp < SSTACK) s_stack[sp][tid] = far; else l_stack[sp - SSTACK] = far;
            ++sp;
          } else if (hl) {
            node = cl;
          } else if (hr) {
            node = cr;
          } else {
            if (sp == 0) break;
            --sp;
            node = sp < SSTACK ? s_stack[sp][tid] : l_stack[sp - SSTACK];
          }
        }
      }

      // ---- oracle step O9: composite the k-buffer front to back, stop at alpha >= 0.99
      bool opaque = false;
#pragma unroll
      for (int i = 0; i < KBUF; ++i) {
        if (!opaque && kb.leaf[i] != EMPTY_LEAF) {
          const float4 col = __ldg(prm.rgba + kb.leaf[i]);
          const float T = sub_(1.0f, A);
          C[0] = fma_(T, col.x, C[0]);
          C[1] = fma_(T, col.y, C[1]);
          C[2] = fma_(T, col.z, C[2]);
          A = fma_(T, col.w, A);
          if (A >= 0.99f) opaque = true;
        }
      }
      if (opaque || !kb.full()) {
        finished = true;
      } else {  // re-launch from the last composited hit
        cur_t = kb.t[KBUF - 1];
        cur_id = __ldg(prm.ids + kb.leaf[KBUF - 1]);
      }
    }
  }
  if (inside) prm.out[(size_t)y * cam.W + x] = make_float4(C[0], C[1], C[2], A);
}

}  // namespace sw
