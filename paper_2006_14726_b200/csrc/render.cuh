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
constexpr int KBUF = 4;
constexpr int SSTACK = 16;
constexpr int LSTACK = 84;  // SSTACK + LSTACK >= 63 key bits + 32 index bits + 1
constexpr uint32_t EMPTY_LEAF = 0xffffffffu;
constexpr uint32_t STACK_DONE = 0xffffffffu;  // not a legal leaf-range code (first < 2^26 - 1)

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
__device__ unsigned long long g_stats[8];  // 0 node visits, 1 sphere tests, 2 hits kept, 3 passes, 4 leaf ranges, 5 max stack
#define STAT_ADD(i, v) atomicAdd(&g_stats[i], (unsigned long long)(v))
#define STAT_MAX(i, v) atomicMax(&g_stats[i], (unsigned long long)(v))
#else
#define STAT_ADD(i, v)
#define STAT_MAX(i, v)
#endif

// The K nearest hits beyond the cursor, sorted by (t, id); alpha rides along so that the
// traversal knows the distance at which the ray becomes opaque.
struct KBuffer {
  float t[KBUF];
  uint32_t leaf[KBUF];
  float al[KBUF];
  __device__ __forceinline__ void clear() {
#pragma unroll
    for (int i = 0; i < KBUF; ++i) { t[i] = __int_as_float(0x7f800000); leaf[i] = EMPTY_LEAF; al[i] = 0.0f; }
  }
  // A full buffer may have dropped hits (evicted here, or culled by the t <= t[K-1] bound).
  __device__ __forceinline__ bool full() const { return leaf[KBUF - 1] != EMPTY_LEAF; }
  // sorted insertion by (t, id); the largest entry falls out when the buffer is full
  __device__ __forceinline__ void insert(float ct, uint32_t cl, float ca, const uint32_t* __restrict__ ids) {
#pragma unroll
    for (int i = 0; i < KBUF; ++i) {
      bool lt = ct < t[i];
      if (!lt && ct == t[i] && leaf[i] != EMPTY_LEAF && cl != EMPTY_LEAF) lt = __ldg(ids + cl) < __ldg(ids + leaf[i]);
      if (lt) {
        const float tt = t[i]; t[i] = ct; ct = tt;
        const uint32_t tl = leaf[i]; leaf[i] = cl; cl = tl;
        const float ta = al[i]; al[i] = ca; ca = ta;
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
  __shared__ uint32_t s_node[SSTACK][RENDER_THREADS];
  __shared__ float s_tn[SSTACK][RENDER_THREADS];
  uint32_t l_node[LSTACK];
  float l_tn[LSTACK];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const DevCamera& cam = prm.cam;
  const int x = blockIdx.x * 16 + (warp & 1) * 8 + (lane & 7);
  const int y = blockIdx.y * 8 + (warp >> 1) * 4 + (lane >> 3);
  const bool inside = x < cam.W && y < cam.H;
  const int n = (int)prm.st->n;
  const float INF = __int_as_float(0x7f800000);

  float o[3] = {cam.e[0], cam.e[1], cam.e[2]};
  float d[3], len;
  pixel_ray(cam, min(x, cam.W - 1), min(y, cam.H - 1), d, len);

  // Conservative slab test (free arithmetic): boxes are padded by far more
  // than the float32 error of ray_sphere(), and the test is one FMA per plane:
  // (plane -+ pad - o) / d = plane * idir - (o +- pad) * idir.
  float m = 1.0f;
#pragma unroll
  for (int a = 0; a < 3; ++a)
    m = fmaxf(m, fmaxf(fabsf(o[a]), fmaxf(fabsf(prm.st->root_lo[a]), fabsf(prm.st->root_hi[a]))));
  const float pad = 4e-5f * m;
  float idir[3], oip[3], oim[3];
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    const float dd = fabsf(d[a]) < 1e-30f ? copysignf(1e-30f, d[a]) : d[a];  // no Inf * 0 in the FMAs
    idir[a] = 1.0f / dd;
    oip[a] = (o[a] + pad) * idir[a];
    oim[a] = (o[a] - pad) * idir[a];
  }

  float C[3] = {0.0f, 0.0f, 0.0f}, A = 0.0f;
  float cur_t = -1.0f;
  uint32_t cur_id = 0;
  bool finished = !inside || n == 0;
  KBuffer kb;

  while (__any_sync(0xffffffffu, !finished)) {
    if (!finished) {
      kb.clear();
      const float t_lo = fmaxf(cur_t, 0.0f);
      float t_hi = INF;  // nothing beyond t_hi can change the pixel: min(k-th hit, opacity cut)
      STAT_ADD(3, 1);

      int sp = 0;
      auto pop = [&]() -> uint32_t {  // next stack entry that is not culled by t_hi
        while (sp > 0) {
          --sp;
          const float tn = sp < SSTACK ? s_tn[sp][tid] : l_tn[sp - SSTACK];
          if (tn <= t_hi) return sp < SSTACK ? s_node[sp][tid] : l_node[sp - SSTACK];
        }
        return STACK_DONE;
      };

      uint32_t node = n == 1 ? leaf_range_code(0u, 1u) : 0u;
      while (true) {
        // ---- internal nodes: both child boxes come with the node (4 x 16-byte loads)
        while ((int)node >= 0) {
          const float4* np = reinterpret_cast<const float4*>(prm.nodes + node);
          const float4 n0 = __ldg(np), n1 = __ldg(np + 1), n2 = __ldg(np + 2), n3 = __ldg(np + 3);
          STAT_ADD(0, 1);
          STAT_MAX(5, sp);
          // left box: lo (n0.x n0.y n0.z) hi (n0.w n1.x n1.y); right box: lo (n1.z n1.w n2.x) hi (n2.y n2.z n2.w)
          float a0 = fmaf(n0.x, idir[0], -oip[0]), a1 = fmaf(n0.w, idir[0], -oim[0]);
          float b0 = fmaf(n0.y, idir[1], -oip[1]), b1 = fmaf(n1.x, idir[1], -oim[1]);
          float c0 = fmaf(n0.z, idir[2], -oip[2]), c1 = fmaf(n1.y, idir[2], -oim[2]);
          const float tnl = fmaxf(fmaxf(fminf(a0, a1), fminf(b0, b1)), fmaxf(fminf(c0, c1), t_lo));
          const float tfl = fminf(fminf(fmaxf(a0, a1), fmaxf(b0, b1)), fminf(fmaxf(c0, c1), t_hi));
          a0 = fmaf(n1.z, idir[0], -oip[0]); a1 = fmaf(n2.y, idir[0], -oim[0]);
          b0 = fmaf(n1.w, idir[1], -oip[1]); b1 = fmaf(n2.z, idir[1], -oim[1]);
          c0 = fmaf(n2.x, idir[2], -oip[2]); c1 = fmaf(n2.w, idir[2], -oim[2]);
          const float tnr = fmaxf(fmaxf(fminf(a0, a1), fminf(b0, b1)), fmaxf(fminf(c0, c1), t_lo));
          const float tfr = fminf(fminf(fmaxf(a0, a1), fmaxf(b0, b1)), fminf(fmaxf(c0, c1), t_hi));
          const bool hl = tnl <= tfl, hr = tnr <= tfr;
          const uint32_t cl = __float_as_uint(n3.x), cr = __float_as_uint(n3.y);
          if (hl && hr) {
            const bool left_first = tnl <= tnr;
            const uint32_t far = left_first ? cr : cl;
            const float tfar = left_first ? tnr : tnl;
            node = left_first ? cl : cr;
            if (sp < SSTACK) { s_node[sp][tid] = far; s_tn[sp][tid] = tfar; }
            else { l_node[sp - SSTACK] = far; l_tn[sp - SSTACK] = tfar; }
            ++sp;
          } else if (hl) {
            node = cl;
          } else if (hr) {
            node = cr;
          } else {
            node = pop();
          }
        }
        if (node == STACK_DONE) break;
        // ---- leaf range: <= LEAF_MAX consecutive splats of the sorted order
        const uint32_t first = leaf_range_first(node), cnt = leaf_range_count(node);
        STAT_ADD(4, 1);
        for (uint32_t j = 0; j < cnt; ++j) {
          const uint32_t leaf = first + j;
          const float4 s = __ldg(prm.sphere + leaf);
          float t;
          STAT_ADD(1, 1);
          if (ray_sphere(o, d, s, t) && t <= t_hi &&
              (t > cur_t || (t == cur_t && __ldg(prm.ids + leaf) > cur_id))) {
            STAT_ADD(2, 1);
            kb.insert(t, leaf, __ldg(&prm.rgba[leaf].w), prm.ids);
            // distance at which the composite below (oracle step O9, same operations in the
            // same order) reaches alpha >= 0.99: later hits cannot contribute
            float a = A, t_cut = INF;
#pragma unroll
            for (int i = 0; i < KBUF; ++i) {
              if (kb.leaf[i] != EMPTY_LEAF && t_cut == INF) {
                a = fma_(sub_(1.0f, a), kb.al[i], a);
                if (a >= 0.99f) t_cut = kb.t[i];
              }
            }
            t_hi = fminf(kb.t[KBUF - 1], t_cut);
          }
        }
        node = pop();
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
