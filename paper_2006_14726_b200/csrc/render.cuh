// render.cuh -- step a6 of SURVEY.md sec. 8(a): per-pixel software BVH traversal of the sphere
// splats with front-to-back compositing of every entry hit ("render them as a point cloud
// using ray tracing"; "spheres that are represented as real quadrics",
// PAPER.md:55; CUDA software ray tracing without RT cores).
//
// One thread per destination pixel, one warp per 8x4 pixel tile, one warp per block (32 resident
// blocks per SM; four consecutive tickets are the four tiles of a 16x8 supertile).  Traversal keeps the K nearest hits beyond a cursor (t, id) in a register
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

constexpr int RENDER_THREADS = 32;   // one warp = one 8x4 tile per block: the finest unit for filling another render's tail
#ifndef SPLATS_KBUF
#define SPLATS_KBUF 4
#endif
constexpr int KBUF = SPLATS_KBUF;
#ifndef SPLATS_SSTACK
#define SPLATS_SSTACK 8
#endif
constexpr int SSTACK = SPLATS_SSTACK;  // deeper entries live in local memory; 8 leaves more of the SM's 256 KB to L1 (4 .. 16 measured: within 1 %)
constexpr int LSTACK = 96 - SSTACK;  // SSTACK + LSTACK >= 63 key bits + 32 index bits + 1
#ifndef SPLATS_POSTPONE
#define SPLATS_POSTPONE 0
#endif
constexpr uint32_t EMPTY_LEAF = 0xffffffffu;
constexpr uint32_t STACK_DONE = 0xffffffffu;  // not a legal leaf-range code (first < 2^26 - 1)

// the image is written once and not read again by this library: streaming stores keep it from
// displacing the BVH in L2
#ifdef SPLATS_OUT_PLAIN
#define OUT_STORE(p, v) (*(p) = (v))
#else
#define OUT_STORE(p, v) __stcs((p), (v))
#endif

struct RenderParams {
  DevCamera cam;
  const QNode* qnodes;   // 32-byte traversal records (common.cuh)
  const float4* sphere;
  const float4* rgba;
  const uint32_t* ids;
  const FrameState* st;
  float4* out;       // float32 RGBA image ...
  uint32_t* out8;    // ... or RGBA8 (OUT8 instances): exactly one of the two is used
  unsigned* sched;  // [0] tile ticket, [1] blocks done (both zero between launches); one pair per render in flight
  int wait_prev;    // 0: this render does not depend on the kernel before it in the stream (see do_render)
  unsigned long long* traced;  // += pixels of the 8x4 tiles inside the scene's screen rectangle (rays set up), once per launch
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
template <int KBUF>
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

// Screen rectangle (in 8x4-pixel warp tiles) that contains every pixel whose ray can touch the
// scene box: the projection of a convex box is the hull of its projected corners.  A corner at
// or behind the eye plane makes the rectangle the whole screen.  Computed by 8 lanes of warp 0.
__device__ __forceinline__ void screen_rect(const DevCamera& cam, const float lo[3], const float hi[3], int lane,
                                            int rect[4]) {
  const int c = lane & 7;
  const float v[3] = {((c & 1) ? hi[0] : lo[0]) - cam.e[0], ((c & 2) ? hi[1] : lo[1]) - cam.e[1],
                      ((c & 4) ? hi[2] : lo[2]) - cam.e[2]};
  const float z = v[0] * cam.F[0] + v[1] * cam.F[1] + v[2] * cam.F[2];
  const float xr = v[0] * cam.R[0] + v[1] * cam.R[1] + v[2] * cam.R[2];
  const float yu = v[0] * cam.U[0] + v[1] * cam.U[1] + v[2] * cam.U[2];
  const bool behind = !(z > 1e-6f * (fabsf(xr) + fabsf(yu) + fabsf(z)) && z > 0.0f);
  // pixel centre x has ndc (2x+1-W)/W; row y has ndc (H-2y-1)/H
  float px = ((xr / (z * cam.ta)) * cam.fW + cam.fW - 1.0f) * 0.5f;
  float py = (cam.fH - 1.0f - (yu / (z * cam.tau)) * cam.fH) * 0.5f;
  float x0 = px, x1 = px, y0 = py, y1 = py;
#pragma unroll
  for (int o = 4; o > 0; o >>= 1) {
    x0 = fminf(x0, __shfl_xor_sync(0xffffffffu, x0, o));
    x1 = fmaxf(x1, __shfl_xor_sync(0xffffffffu, x1, o));
    y0 = fminf(y0, __shfl_xor_sync(0xffffffffu, y0, o));
    y1 = fmaxf(y1, __shfl_xor_sync(0xffffffffu, y1, o));
  }
  const bool any_behind = __any_sync(0xffffffffu, behind);
  const int tiles_x = (cam.W + 7) >> 3, tiles_y = (cam.H + 3) >> 2;
  if (any_behind || !(x0 == x0) || !(x1 == x1) || !(y0 == y0) || !(y1 == y1)) {
    rect[0] = 0; rect[1] = 0; rect[2] = (tiles_x + 1) & ~1; rect[3] = (tiles_y + 1) & ~1;
    return;
  }
  // two pixels of slack: far more than the float32 error of the projection above
  const float fx0 = fmaxf(floorf(x0) - 2.0f, 0.0f), fx1 = fminf(ceilf(x1) + 2.0f, cam.fW - 1.0f);
  const float fy0 = fmaxf(floorf(y0) - 2.0f, 0.0f), fy1 = fminf(ceilf(y1) + 2.0f, cam.fH - 1.0f);
  if (fx0 > fx1 || fy0 > fy1) { rect[0] = rect[1] = rect[2] = rect[3] = 0; return; }  // off screen
  rect[0] = ((int)fx0 >> 4) << 1; rect[1] = ((int)fy0 >> 3) << 1;   // aligned to 16x8-pixel supertiles
  rect[2] = (((int)fx1 >> 4) + 1) << 1; rect[3] = (((int)fy1 >> 3) + 1) << 1;   // exclusive
}

// Persistent grid (SMs x resident blocks).  (A) every pixel outside the scene's screen rectangle
// is background: written as zeros by a grid-stride loop, no ray is set up for it.  (B) the 8x4
// warp tiles inside the rectangle are handed out dynamically: a warp's first tile is its index
// in the grid, every further one comes from an atomic ticket; the last block to finish re-arms
// the ticket for the next launch.
//
// FIRST = true is the paper's own query ("a simple first-hit ray tracing query and
// with no shading other than the constant sample color"): a one-entry buffer keeps the nearest
// hit in (t, id) order, everything beyond it is culled, and its stored colour is copied out.
// OUT8 = true writes the pixel as RGBA8 (round(255 c), the colour format of the wire, S10) instead
// of four float32: a quarter of the bytes for a client that only displays the image.
template <int KBUF, bool FIRST, bool OUT8 = false>
#ifndef SPLATS_RENDER_BLOCKS
#define SPLATS_RENDER_BLOCKS (1024 / RENDER_THREADS)
#endif
__global__ void __launch_bounds__(RENDER_THREADS, SPLATS_RENDER_BLOCKS)
render_kernel(RenderParams prm) {
  if (prm.wait_prev) pdl_wait();
  pdl_trigger();
  // stack entry = (node, entry distance) as one 8-byte word; [depth][thread]: conflict free.  Addressed through
  // one precomputed shared-memory address (the compiler otherwise rebuilds it at every push and pop).
  __shared__ uint2 s_stack[SSTACK][RENDER_THREADS];
  __shared__ int s_rect[4];
  uint32_t l_node[LSTACK];
  float l_tn[LSTACK];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  uint32_t s_base;   // opaque to the compiler, or it is rematerialised (thread id, CTA id, shifts) at every use
  asm volatile("mov.u32 %0, %1;" : "=r"(s_base) : "r"((uint32_t)__cvta_generic_to_shared(&s_stack[0][tid])));
  constexpr uint32_t S_STRIDE = RENDER_THREADS * sizeof(uint2);
  const DevCamera& cam = prm.cam;
  const int n = (int)prm.st->n;
  const float INF = __int_as_float(0x7f800000);
  const float o[3] = {cam.e[0], cam.e[1], cam.e[2]};

  // conservative padding of every box: far more than the float32 error of ray_sphere()
  float m = 1.0f;
#pragma unroll
  for (int a = 0; a < 3; ++a)
    m = fmaxf(m, fmaxf(fabsf(o[a]), fmaxf(fabsf(prm.st->root_lo[a]), fabsf(prm.st->root_hi[a]))));
  const float pad = 4e-5f * m;
  const QFrame qf = load_qframe(prm.st);

  if (warp == 0) {
    int rect[4] = {0, 0, 0, 0};
    if (n > 0) {
      const float lo[3] = {prm.st->root_lo[0] - pad, prm.st->root_lo[1] - pad, prm.st->root_lo[2] - pad};
      const float hi[3] = {prm.st->root_hi[0] + pad, prm.st->root_hi[1] + pad, prm.st->root_hi[2] + pad};
      screen_rect(cam, lo, hi, lane, rect);
    }
    if (lane < 4) s_rect[lane] = rect[lane];
  }
  __syncthreads();
  const int rx0 = s_rect[0], ry0 = s_rect[1], rx1 = s_rect[2], ry1 = s_rect[3];

  // ---- (B) warp tiles inside the rectangle
  // tickets [0, ntiles): trace one 8x4 tile (2x2 tiles = one 16x8 supertile are consecutive);
  // tickets [ntiles, ntiles + nfill): zero FILL_PX background pixels outside the rectangle
  constexpr int FILL_PX = 1024;
  const int rw = rx1 - rx0, ntiles = rw * (ry1 - ry0);
  const int total_px = cam.W * cam.H;
  const int nfill = (total_px + FILL_PX - 1) / FILL_PX;
  const int nwarps = gridDim.x * (RENDER_THREADS / 32);
  if (blockIdx.x == 0 && tid == 0) atomicAdd(prm.traced, (unsigned long long)ntiles * 32ull);
  int tile = blockIdx.x * (RENDER_THREADS / 32) + warp;
  for (; tile < ntiles + nfill; tile = nwarps + (int)__shfl_sync(0xffffffffu, lane == 0 ? atomicAdd(prm.sched, 1u) : 0u, 0)) {
  if (tile >= ntiles) {
    const int px0 = rx0 * 8, px1 = rx1 * 8, py0 = ry0 * 4, py1 = ry1 * 4;
    const int base = (tile - ntiles) * FILL_PX;
#pragma unroll 4
    for (int k = lane; k < FILL_PX; k += 32) {
      const int idx = base + k;
      const int yy = idx / cam.W, xx = idx - yy * cam.W;
      if (idx < total_px && !(xx >= px0 && xx < px1 && yy >= py0 && yy < py1))
        if (OUT8) __stcs(prm.out8 + idx, 0u);
        else OUT_STORE(prm.out + idx, make_float4(0.0f, 0.0f, 0.0f, 0.0f));
    }
    continue;
  }
  // The rectangle is aligned to supertiles.  Supertile rows are handed out from the middle of
  // the rectangle outwards (mid, mid-1, mid+1, ...): the rows that are likely to hold the most
  // hits start first and the kernel's tail is made of the cheap rows at the top and bottom edge.
  const int sw = rw >> 1, sh = (ry1 - ry0) >> 1, super = tile >> 2;
  const int rr = super / sw;
  const int srow = (sh >> 1) + ((rr & 1) ? -((rr + 1) >> 1) : (rr >> 1));
  const int ty = srow * 2 + ((tile >> 1) & 1), tx = (super - rr * sw) * 2 + (tile & 1);
  const int x = (rx0 + tx) * 8 + (lane & 7);
  const int y = (ry0 + ty) * 4 + (lane >> 3);
  const bool inside = x < cam.W && y < cam.H;

  float d[3], len;
  pixel_ray(cam, min(x, cam.W - 1), min(y, cam.H - 1), d, len);

  // Conservative slab test (free arithmetic).  A plane of a child box is stored as a 16-bit code q
  // (plane = qf.lo + q qf.c, S13); as_float(0x4B000000 | q) = 2^23 + q exactly, so
  //   t = (plane -+ pad - o) / d = (2^23 + q) * (c / d) + ((qf.lo - o) / d -+ pad / |d| - 2^23 c / d)
  // is ONE byte permute + ONE FMA per plane, and the permute also picks the near / far plane of the
  // axis by the sign of d (no min / max per axis).  The constant's rounding error is half a code
  // step in plane units, so the box is padded by one more step than the exact boxes were.
  float qa[3], bn[3], bf[3];
  uint32_t seln[3], self[3];
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    const float dd = fabsf(d[a]) < 1e-30f ? copysignf(1e-30f, d[a]) : d[a];  // no Inf * 0 in the FMAs
    const float idir = 1.0f / dd;
    qa[a] = qf.c[a] * idir;
    const float b0 = fmaf(-8388608.0f, qa[a], (qf.lo[a] - o[a]) * idir), pd = (pad + qf.c[a]) * fabsf(idir);
    bn[a] = b0 - pd;
    bf[a] = b0 + pd;
    seln[a] = dd >= 0.0f ? 0x7610u : 0x7632u;   // low half = lower plane, high half = upper plane
    self[a] = dd >= 0.0f ? 0x7632u : 0x7610u;
  }

  float C[3] = {0.0f, 0.0f, 0.0f}, A = 0.0f;
  float cur_t = -1.0f;
  uint32_t cur_id = 0;
  bool finished = !inside;
  KBuffer<KBUF> kb;

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
          uint32_t nd;
          float tn;
          if (sp < SSTACK) asm volatile("ld.shared.v2.b32 {%0, %1}, [%2];" : "=r"(nd), "=f"(tn) : "r"(s_base + sp * S_STRIDE));
          else { nd = l_node[sp - SSTACK]; tn = l_tn[sp - SSTACK]; }
          if (tn <= t_hi) return nd;
        }
        return STACK_DONE;
      };

      uint32_t node = n == 1 ? leaf_range_code(0u, 1u) : 0u, pend = STACK_DONE;
      while (true) {
        // ---- internal nodes: both child boxes come with the node (one 32-byte load)
        while ((int)node >= 0) {
          const u8x rec = ldg_u8(prm.qnodes + node);
          STAT_ADD(0, 1);
          STAT_MAX(5, sp);
#define QPLANE(w, sel) __uint_as_float(__byte_perm((w), 0x4B000000u, (sel)))
          const float tnl = fmaxf(fmaxf(fmaf(QPLANE(rec.v[0], seln[0]), qa[0], bn[0]), fmaf(QPLANE(rec.v[1], seln[1]), qa[1], bn[1])),
                                  fmaxf(fmaf(QPLANE(rec.v[2], seln[2]), qa[2], bn[2]), t_lo));
          const float tfl = fminf(fminf(fmaf(QPLANE(rec.v[0], self[0]), qa[0], bf[0]), fmaf(QPLANE(rec.v[1], self[1]), qa[1], bf[1])),
                                  fminf(fmaf(QPLANE(rec.v[2], self[2]), qa[2], bf[2]), t_hi));
          const float tnr = fmaxf(fmaxf(fmaf(QPLANE(rec.v[3], seln[0]), qa[0], bn[0]), fmaf(QPLANE(rec.v[4], seln[1]), qa[1], bn[1])),
                                  fmaxf(fmaf(QPLANE(rec.v[5], seln[2]), qa[2], bn[2]), t_lo));
          const float tfr = fminf(fminf(fmaf(QPLANE(rec.v[3], self[0]), qa[0], bf[0]), fmaf(QPLANE(rec.v[4], self[1]), qa[1], bf[1])),
                                  fminf(fmaf(QPLANE(rec.v[5], self[2]), qa[2], bf[2]), t_hi));
#undef QPLANE
          const bool hl = tnl <= tfl, hr = tnr <= tfr;
          const uint32_t cl = rec.v[6], cr = rec.v[7];
          bool need_pop = false;
          if (hl && hr) {
            const bool left_first = tnl <= tnr;
            const uint32_t far = left_first ? cr : cl;
            const float tfar = left_first ? tnr : tnl;
            node = left_first ? cl : cr;
            if (sp < SSTACK) asm volatile("st.shared.v2.b32 [%0], {%1, %2};" :: "r"(s_base + sp * S_STRIDE), "r"(far), "f"(tfar) : "memory");
            else { l_node[sp - SSTACK] = far; l_tn[sp - SSTACK] = tfar; }
            ++sp;
          } else if (hl) {
            node = cl;
          } else if (hr) {
            node = cr;
          } else {
            need_pop = true;
          }
#if SPLATS_POSTPONE
          // a lane that reaches its first leaf keeps it for later and goes on with the next stack entry: the warp
          // stays in this loop together for longer and tests two leaves per lane in the phase below
          if (!need_pop && (int)node < 0 && pend == STACK_DONE) { pend = node; need_pop = true; }
#endif
          if (need_pop) node = pop();
        }
        // ---- leaves: the postponed one, then the one the descent stopped at (<= LEAF_MAX consecutive splats each)
#pragma unroll 1
        for (int which = SPLATS_POSTPONE ? 0 : 1; which < 2; ++which) {
          const uint32_t code = which == 0 ? pend : node;
          if (code == STACK_DONE) continue;
          const uint32_t first = leaf_range_first(code), cnt = leaf_range_count(code);
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
              if (FIRST) {
                t_hi = kb.t[0];  // nothing beyond the nearest hit so far matters
              } else {
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
          }
        }
        pend = STACK_DONE;
        if (node == STACK_DONE) break;
        node = pop();
      }

      if (FIRST) {  // copy the colour of the nearest hit; one traversal is always enough
        if (kb.leaf[0] != EMPTY_LEAF) {
          const float4 col = __ldg(prm.rgba + kb.leaf[0]);
          C[0] = col.x; C[1] = col.y; C[2] = col.z; A = col.w;
        }
        finished = true;
        continue;
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
  if (inside) {
    if (OUT8) __stcs(prm.out8 + (size_t)y * cam.W + x, pack_colour(make_float4(C[0], C[1], C[2], A)));
    else OUT_STORE(prm.out + (size_t)y * cam.W + x, make_float4(C[0], C[1], C[2], A));
  }
  }  // tile loop
  __syncthreads();
  if (tid == 0) {
    __threadfence();
    if (atomicInc(prm.sched + 1, gridDim.x - 1) == gridDim.x - 1) {
      prm.sched[0] = 0u;
      // A render that did not wait for its predecessor at the start must not COMPLETE before it:
      // whatever comes next in the stream (a copy of an earlier image, an event, the next
      // update) orders itself after the last kernel only, so completion has to stay in launch
      // order.  One thread of the last block to finish holds the grid open; every other block
      // exits and frees its slot at once.
      if (!prm.wait_prev) pdl_wait();
    }
  }
}

}  // namespace sw
