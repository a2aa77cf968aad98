// lbvh.cuh -- steps a4 (Karras-style hierarchy emission) and a5 (bottom-up refit with atomic
// arrival counters) of SURVEY.md sec. 8(a), plus the canonical export used by the parity
// tests.  "build a bounding volume hierarchy ... using the LBVH algorithm".
#pragma once
#include "common.cuh"

namespace sw {

constexpr int LBVH_THREADS = 256;

// Splat `id` (= source pixel index, or position in a received sample buffer) as sphere + colour.
// FrameGather recomputes the sphere from the depth buffer with exactly the arithmetic of the
// bounds / Morton kernels (Eq. 1; radius per RadiusParams) and copies the colour
// ("no shading other than the constant sample color"); PackedGather decodes the
// 64-bit sample and the RGBA8 colour.
struct FrameGather {
  const float* __restrict__ depth;
  const float4* __restrict__ color;
  DevCamera cam;
  RadiusParams rp;
  __device__ __forceinline__ void get(uint32_t id, float4& sp, float4& col) const {
    const int y = (int)(id / (uint32_t)cam.W), x = (int)(id - (uint32_t)y * (uint32_t)cam.W);
    const float t = __ldg(depth + id);
    float p[3], len;
    splat_centre(cam, x, y, t, p, len);
    const float z = div_(t, len);
    col = __ldg(color + id);
    sp = make_float4(p[0], p[1], p[2], splat_radius(rp, z, col.w));
  }
};
struct PackedGather {
  const uint64_t* __restrict__ samples;
  const uint32_t* __restrict__ colours;
  QuantParams q;
  __device__ __forceinline__ void get(uint32_t id, float4& sp, float4& col) const {
    const uint64_t w = __ldg(samples + id);
    float p[3];
    decode_centre(w, q, p);
    sp = make_float4(p[0], p[1], p[2], decode_radius(w, q));
    col = decode_colour(__ldg(colours + id));
  }
};

// Common-prefix length of the keys at sorted positions i and j; ties broken by the sorted
// position itself (equivalent to concatenating key and index); -1 outside the array.
__device__ __forceinline__ int delta(const uint64_t* __restrict__ keys, int n, int i, uint64_t ki, int j) {
  if (j < 0 || j >= n) return -1;
  const uint64_t x = ki ^ __ldg(keys + j);
  return x ? __clzll((long long)x) : 64 + __clz(i ^ j);
}

// Thread i (grid-stride): (a) gathers splat perm[i] into sorted order -- the sphere is
// recomputed from the depth buffer with exactly the arithmetic of the bounds/Morton
// kernels (Eq. 1; radius = k_r * view-axis depth), the colour is copied
// ("no shading other than the constant sample color"); (b) emits internal
// node i of the binary radix tree over the sorted keys: direction, range end by
// doubling + binary search, split by binary search.
template <class Gather>
__global__ void __launch_bounds__(LBVH_THREADS)
emit_kernel(const uint64_t* __restrict__ keys, const uint32_t* __restrict__ perm, const Gather src,
            const FrameState* __restrict__ st, float4* __restrict__ sphere, float4* __restrict__ rgba,
            uint32_t* __restrict__ ids_out, Node* __restrict__ nodes, int* __restrict__ leaf_parent) {
  const int n = (int)st->n;
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
    // ---- (a) gather
    float4 sp, col;
    const uint32_t id = __ldg(perm + i);
    src.get(id, sp, col);
    sphere[i] = sp;
    rgba[i] = col;
    ids_out[i] = id;   // the BVH keeps its own copy: the sort buffers belong to the next build
    if (n == 1) leaf_parent[0] = -1;
    if (i >= n - 1) continue;

    // ---- (b) internal node i
    const uint64_t ki = __ldg(keys + i);
    const int d = delta(keys, n, i, ki, i + 1) > delta(keys, n, i, ki, i - 1) ? 1 : -1;
    const int dmin = delta(keys, n, i, ki, i - d);
    int lmax = 2;
    while (delta(keys, n, i, ki, i + lmax * d) > dmin) lmax <<= 1;
    int l = 0;
    for (int t2 = lmax >> 1; t2 >= 1; t2 >>= 1)
      if (delta(keys, n, i, ki, i + (l + t2) * d) > dmin) l += t2;
    const int j = i + l * d;
    const int dnode = delta(keys, n, i, ki, j);
    int s = 0;
    for (int t2 = l; t2 > 1;) {
      t2 = (t2 + 1) >> 1;
      if (delta(keys, n, i, ki, i + (s + t2) * d) > dnode) s += t2;
    }
    const int gamma = i + s * d + min(d, 0);
    const int first = min(i, j), last = max(i, j);
    const bool leaf_l = first == gamma, leaf_r = last == gamma + 1;
    const int cnt_l = gamma - first + 1, cnt_r = last - gamma;
    nodes[i].left = cnt_l <= LEAF_MAX ? (int)leaf_range_code((uint32_t)first, (uint32_t)cnt_l) : gamma;
    nodes[i].right = cnt_r <= LEAF_MAX ? (int)leaf_range_code((uint32_t)gamma + 1u, (uint32_t)cnt_r) : gamma + 1;
    nodes[i].flag = 0u;
    if (i == 0) nodes[0].parent = -1;
    if (leaf_l) leaf_parent[gamma] = (i << 1); else nodes[gamma].parent = (i << 1);
    if (leaf_r) leaf_parent[gamma + 1] = (i << 1) | 1; else nodes[gamma + 1].parent = (i << 1) | 1;
  }
}

// One thread per leaf climbs towards the root.  At every internal node it stores the box it
// carries into the parent's slot for that child, publishes it (fence) and bumps the node's
// arrival counter; the first arrival stops, the second one reads its sibling's slot, forms
// the exact union (fmin/fmax) and continues.  Every internal node is completed exactly once.
__global__ void __launch_bounds__(LBVH_THREADS)
refit_kernel(const float4* __restrict__ sphere, const int* __restrict__ leaf_parent, Node* nodes,
             FrameState* st) {
  const int n = (int)st->n;
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
    const float4 sp = sphere[i];
    float lo[3] = {sub_(sp.x, sp.w), sub_(sp.y, sp.w), sub_(sp.z, sp.w)};
    float hi[3] = {add_(sp.x, sp.w), add_(sp.y, sp.w), add_(sp.z, sp.w)};
    int link = leaf_parent[i];
    while (link >= 0) {
      const int p = link >> 1, side = link & 1;
      float2* slot = reinterpret_cast<float2*>(nodes[p].b + 6 * side);
      __stcg(slot + 0, make_float2(lo[0], lo[1]));
      __stcg(slot + 1, make_float2(lo[2], hi[0]));
      __stcg(slot + 2, make_float2(hi[1], hi[2]));
      __threadfence();
      if (atomicAdd(&nodes[p].flag, 1u) == 0u) break;  // sibling subtree not finished yet
      __threadfence();
      const float2* other = reinterpret_cast<const float2*>(nodes[p].b + 6 * (side ^ 1));
      const float2 a = __ldcg(other + 0), b = __ldcg(other + 1), c = __ldcg(other + 2);
      lo[0] = fminf(lo[0], a.x); lo[1] = fminf(lo[1], a.y); lo[2] = fminf(lo[2], b.x);
      hi[0] = fmaxf(hi[0], b.y); hi[1] = fmaxf(hi[1], c.x); hi[2] = fmaxf(hi[2], c.y);
      link = __ldcg(&nodes[p].parent);
    }
    if (link < 0) {  // this thread completed the root (or is the single leaf): scene box
#pragma unroll
      for (int a = 0; a < 3; ++a) { st->root_lo[a] = lo[a]; st->root_hi[a] = hi[a]; }
    }
  }
}

// ===================================================================== pyramid refit
// The default a4/a5 path (splats_set_option(SPLATS_OPT_REFIT, SPLATS_REFIT_PYRAMID)).
//
// A node of the radix tree covers a contiguous range of the sorted leaves, so its box is a
// range min/max over the leaf boxes.  Instead of climbing the tree with one fence + atomic
// per level (a dependent chain as long as the tree is deep), (1) leaf_pyramid_kernel gathers
// the splats into sorted order and builds a binary min/max pyramid over the leaf boxes --
// bottom-up, ten levels per block in shared memory, the remaining ones by the last block to
// finish --, (2) hierarchy_kernel finds the range and split of every node i (Karras) beside it,
// and (3) boxes_kernel obtains both child boxes of a node by a range query on the pyramid
// (<= 2 log2(range) independent entry reads, no atomics, no fences).
// min/max are exact and associative, so the boxes are bit-identical to a bottom-up refit.
constexpr int PYR_THREADS = 256;
constexpr int PYR_LEAVES = 1024;     // leaves per block = 2^PYR_LOCAL
constexpr int PYR_LOCAL = 10;
constexpr int PYR_MAX_LEVELS = 27;   // capacity < 2^26 leaves

// Level k >= 1 holds ceil(cap / 2^k) entries of two float4 (lo xyz, hi xyz) starting at entry
// off[k]; entry j of level k is the box of the leaves [j 2^k, (j+1) 2^k) that exist.
struct PyramidLayout {
  uint32_t off[PYR_MAX_LEVELS + 1];
};
__constant__ PyramidLayout c_pyr;   // set once in splats_create (indexed by a run-time level)

__device__ __forceinline__ void box_of_sphere(const float4 sp, float lo[3], float hi[3]) {
  lo[0] = sub_(sp.x, sp.w); lo[1] = sub_(sp.y, sp.w); lo[2] = sub_(sp.z, sp.w);
  hi[0] = add_(sp.x, sp.w); hi[1] = add_(sp.y, sp.w); hi[2] = add_(sp.z, sp.w);
}

template <class Gather>
__global__ void __launch_bounds__(PYR_THREADS)
leaf_pyramid_kernel(const uint32_t* __restrict__ perm, const Gather src, FrameState* st,
                    float4* __restrict__ sphere, float4* __restrict__ rgba, uint32_t* __restrict__ ids_out, float4* pyr) {
  pdl_wait();
  pdl_trigger();
  __shared__ float s_box[6][PYR_LEAVES];
  __shared__ bool s_last;
  const uint32_t n = st->n;
  const uint32_t nblocks = (n + PYR_LEAVES - 1) / PYR_LEAVES;
  if (blockIdx.x >= nblocks) return;
  const int tid = threadIdx.x;
  const uint32_t base = blockIdx.x * PYR_LEAVES;
  const float INF = __int_as_float(0x7f800000);

  // ---- gather the splats of this block into sorted order; leaf boxes -> shared memory
#pragma unroll
  for (int j = 0; j < PYR_LEAVES / PYR_THREADS; ++j) {
    const int l = tid + j * PYR_THREADS;
    const uint32_t i = base + l;
    float lo[3] = {INF, INF, INF}, hi[3] = {-INF, -INF, -INF};
    if (i < n) {
      float4 sp, col;
      const uint32_t id = __ldg(perm + i);
      src.get(id, sp, col);
      sphere[i] = sp;
      rgba[i] = col;
      ids_out[i] = id;   // the BVH keeps its own copy: the sort buffers belong to the next build
      box_of_sphere(sp, lo, hi);
    }
#pragma unroll
    for (int a = 0; a < 3; ++a) { s_box[a][l] = lo[a]; s_box[3 + a][l] = hi[a]; }
  }
  __syncthreads();

  // ---- levels 1..PYR_LOCAL, in place: level k entry j ends up in s_box[.][j]
#pragma unroll
  for (int k = 1; k <= PYR_LOCAL; ++k) {
    const int cnt = PYR_LEAVES >> k;
    float v[2][6];
#pragma unroll
    for (int r = 0; r < 2; ++r) {
      const int j = tid + r * PYR_THREADS;
      if (j < cnt) {
#pragma unroll
        for (int a = 0; a < 3; ++a) {
          v[r][a] = fminf(s_box[a][2 * j], s_box[a][2 * j + 1]);
          v[r][3 + a] = fmaxf(s_box[3 + a][2 * j], s_box[3 + a][2 * j + 1]);
        }
      }
    }
    __syncthreads();
#pragma unroll
    for (int r = 0; r < 2; ++r) {
      const int j = tid + r * PYR_THREADS;
      if (j < cnt) {
#pragma unroll
        for (int a = 0; a < 6; ++a) s_box[a][j] = v[r][a];
        if (base + ((uint32_t)j << k) < n) {
          float4* e = pyr + 2 * ((size_t)c_pyr.off[k] + (base >> k) + j);
          __stcg(e, make_float4(v[r][0], v[r][1], v[r][2], 0.0f));
          __stcg(e + 1, make_float4(v[r][3], v[r][4], v[r][5], 0.0f));
        }
      }
    }
    __syncthreads();
  }
  if (nblocks == 1) return;

  // ---- the last block to finish builds the levels above PYR_LOCAL
  __threadfence();
  if (tid == 0) s_last = atomicAdd(&st->pyr_done, 1u) == nblocks - 1;
  __syncthreads();
  if (!s_last) return;
  __threadfence();
  uint32_t cnt_prev = nblocks;
  for (int k = PYR_LOCAL + 1; cnt_prev > 1; ++k) {
    const uint32_t cnt = (cnt_prev + 1) >> 1;
    const float4* src = pyr + 2 * (size_t)c_pyr.off[k - 1];
    float4* dst = pyr + 2 * (size_t)c_pyr.off[k];
    for (uint32_t j = tid; j < cnt; j += PYR_THREADS) {
      float4 lo = __ldcg(src + 4 * (size_t)j), hi = __ldcg(src + 4 * (size_t)j + 1);
      if (2 * j + 1 < cnt_prev) {
        const float4 lo2 = __ldcg(src + 4 * (size_t)j + 2), hi2 = __ldcg(src + 4 * (size_t)j + 3);
        lo.x = fminf(lo.x, lo2.x); lo.y = fminf(lo.y, lo2.y); lo.z = fminf(lo.z, lo2.z);
        hi.x = fmaxf(hi.x, hi2.x); hi.y = fmaxf(hi.y, hi2.y); hi.z = fmaxf(hi.z, hi2.z);
      }
      __stcg(dst + 2 * (size_t)j, lo);
      __stcg(dst + 2 * (size_t)j + 1, hi);
    }
    __syncthreads();
    cnt_prev = cnt;
  }
}

// Boxes of the sorted leaves [l0, r0) and [l1, r1) (l < r <= n): two iterative segment-tree
// queries in lockstep, level 0 read from the spheres, every other level from the pyramid.  The
// entry addresses do not depend on loaded data, so the loads of level k+1 are issued before the
// entries of level k are consumed (software pipelining: the kernel is latency bound).
struct BoxAcc {
  float lo[3], hi[3];
  __device__ __forceinline__ void init() {
    const float INF = __int_as_float(0x7f800000);
#pragma unroll
    for (int a = 0; a < 3; ++a) { lo[a] = INF; hi[a] = -INF; }
  }
  __device__ __forceinline__ void add(const float4 a, const float4 b) {
    lo[0] = fminf(lo[0], a.x); lo[1] = fminf(lo[1], a.y); lo[2] = fminf(lo[2], a.z);
    hi[0] = fmaxf(hi[0], b.x); hi[1] = fmaxf(hi[1], b.y); hi[2] = fmaxf(hi[2], b.z);
  }
  __device__ __forceinline__ void add_sphere(const float4 sp) {
    float blo[3], bhi[3];
    box_of_sphere(sp, blo, bhi);
#pragma unroll
    for (int a = 0; a < 3; ++a) { lo[a] = fminf(lo[a], blo[a]); hi[a] = fmaxf(hi[a], bhi[a]); }
  }
};

__device__ __forceinline__ void range_box2(const float4* __restrict__ sphere, const float4* __restrict__ pyr,
                                           uint32_t l0, uint32_t r0, uint32_t l1, uint32_t r1, BoxAcc& A, BoxAcc& B) {
  A.init();
  B.init();
  uint32_t l[2] = {l0, l1}, r[2] = {r0, r1};
  const float4 Z = make_float4(0.f, 0.f, 0.f, 0.f);
  float4 ea[4], eb[4];  // pending entries: [2 q + side]
  bool pend[4];
  {  // level 0: spheres
    float4 s[4];
#pragma unroll
    for (int q = 0; q < 2; ++q) {
      pend[2 * q] = l[q] & 1u;
      pend[2 * q + 1] = r[q] & 1u;
      s[2 * q] = pend[2 * q] ? __ldg(sphere + l[q]) : Z;
      s[2 * q + 1] = pend[2 * q + 1] ? __ldg(sphere + r[q] - 1) : Z;
      l[q] = (l[q] + 1) >> 1;
      r[q] >>= 1;
    }
    if (pend[0]) A.add_sphere(s[0]);
    if (pend[1]) A.add_sphere(s[1]);
    if (pend[2]) B.add_sphere(s[2]);
    if (pend[3]) B.add_sphere(s[3]);
  }
#pragma unroll
  for (int e = 0; e < 4; ++e) { pend[e] = false; ea[e] = Z; eb[e] = Z; }
  for (int k = 1; l[0] < r[0] || l[1] < r[1]; ++k) {
    const float4* lev = pyr + 2 * (size_t)c_pyr.off[k];
    float4 na[4], nb[4];
    bool np[4];
#pragma unroll
    for (int q = 0; q < 2; ++q) {
      const bool act = l[q] < r[q];
      np[2 * q] = act && (l[q] & 1u);
      np[2 * q + 1] = act && (r[q] & 1u);
      na[2 * q] = np[2 * q] ? __ldg(lev + 2 * (size_t)l[q]) : Z;
      nb[2 * q] = np[2 * q] ? __ldg(lev + 2 * (size_t)l[q] + 1) : Z;
      na[2 * q + 1] = np[2 * q + 1] ? __ldg(lev + 2 * (size_t)(r[q] - 1)) : Z;
      nb[2 * q + 1] = np[2 * q + 1] ? __ldg(lev + 2 * (size_t)(r[q] - 1) + 1) : Z;
      l[q] = (l[q] + 1) >> 1;
      r[q] >>= 1;
    }
    if (pend[0]) A.add(ea[0], eb[0]);
    if (pend[1]) A.add(ea[1], eb[1]);
    if (pend[2]) B.add(ea[2], eb[2]);
    if (pend[3]) B.add(ea[3], eb[3]);
#pragma unroll
    for (int e = 0; e < 4; ++e) { pend[e] = np[e]; ea[e] = na[e]; eb[e] = nb[e]; }
  }
  if (pend[0]) A.add(ea[0], eb[0]);
  if (pend[1]) A.add(ea[1], eb[1]);
  if (pend[2]) B.add(ea[2], eb[2]);
  if (pend[3]) B.add(ea[3], eb[3]);
}

// Largest x in [base, base + width) with delta(i, i + x d) > dref, given that it holds at
// `base` and fails at base + width (width a power of two; the predicate is monotone because
// the common prefix with key i can only shrink with distance).  Two bits per step from three
// independent probes: half the dependent loads of a binary search.
__device__ __forceinline__ int descend4(const uint64_t* __restrict__ keys, int n, int i, uint64_t ki, int d,
                                        int dref, int base, int width) {
  while (width >= 4) {
    const int q = width >> 2;
    const int c = (int)(delta(keys, n, i, ki, i + (base + q) * d) > dref) +
                  (int)(delta(keys, n, i, ki, i + (base + 2 * q) * d) > dref) +
                  (int)(delta(keys, n, i, ki, i + (base + 3 * q) * d) > dref);
    base += c * q;
    width = q;
  }
  if (width == 2 && delta(keys, n, i, ki, i + (base + 1) * d) > dref) base += 1;
  return base;
}

// Internal node i of the binary radix tree (Karras: direction, range end by galloping + search,
// split by search): the sorted leaves it covers, [first, last], and its split gamma (left child
// covers [first, gamma]).
__device__ __forceinline__ void karras_node(const uint64_t* __restrict__ keys, int n, int i, int& first, int& gamma,
                                            int& last) {
  const uint64_t ki = __ldg(keys + i);
  const int d = delta(keys, n, i, ki, i + 1) > delta(keys, n, i, ki, i - 1) ? 1 : -1;
  const int dmin = delta(keys, n, i, ki, i - d);
  // gallop: the range length l satisfies lb <= l < 2 lb (four probes per round)
  int lb = 1;
  while (true) {
    const int c = (int)(delta(keys, n, i, ki, i + 2 * lb * d) > dmin) + (int)(delta(keys, n, i, ki, i + 4 * lb * d) > dmin) +
                  (int)(delta(keys, n, i, ki, i + 8 * lb * d) > dmin) + (int)(delta(keys, n, i, ki, i + 16 * lb * d) > dmin);
    lb <<= c;
    if (c < 4) break;
  }
  const int l = descend4(keys, n, i, ki, d, dmin, lb, lb);
  const int j = i + l * d;
  const int dnode = delta(keys, n, i, ki, j);
  // split: largest s in [0, l) whose key still shares more than dnode bits with key i
  const int s = descend4(keys, n, i, ki, d, dnode, 0, l > 1 ? 1 << (32 - __clz(l - 1)) : 1);
  gamma = i + s * d + min(d, 0);
  first = min(i, j);
  last = max(i, j);
}

// The 64-byte record of node i: both child boxes as range queries on the pyramid, child links.
__device__ __forceinline__ void write_node(const float4* __restrict__ sphere, const float4* __restrict__ pyr, FrameState* st,
                                           Node* __restrict__ nodes, int i, int first, int gamma, int last) {
  const int cnt_l = gamma - first + 1, cnt_r = last - gamma;
  BoxAcc L, R;
  range_box2(sphere, pyr, (uint32_t)first, (uint32_t)gamma + 1u, (uint32_t)gamma + 1u, (uint32_t)last + 1u, L, R);
  const int left = cnt_l <= LEAF_MAX ? (int)leaf_range_code((uint32_t)first, (uint32_t)cnt_l) : gamma;
  const int right = cnt_r <= LEAF_MAX ? (int)leaf_range_code((uint32_t)gamma + 1u, (uint32_t)cnt_r) : gamma + 1;
  float4* rec = reinterpret_cast<float4*>(nodes + i);
  rec[0] = make_float4(L.lo[0], L.lo[1], L.lo[2], L.hi[0]);
  rec[1] = make_float4(L.hi[1], L.hi[2], R.lo[0], R.lo[1]);
  rec[2] = make_float4(R.lo[2], R.hi[0], R.hi[1], R.hi[2]);
  rec[3] = make_float4(__int_as_float(left), __int_as_float(right), 0.0f, 0.0f);
  if (i == 0) {
#pragma unroll
    for (int a = 0; a < 3; ++a) { st->root_lo[a] = fminf(L.lo[a], R.lo[a]); st->root_hi[a] = fmaxf(L.hi[a], R.hi[a]); }
  }
}

// The hierarchy needs only the sorted keys, the pyramid only the sorted ids: hierarchy_kernel
// runs beside leaf_pyramid_kernel (it is launched as a programmatic dependent that does not wait
// for it at the start but at the end, so that the kernel after it is ordered after both), and
// boxes_kernel then joins the two: ranges + pyramid -> node records.
__global__ void __launch_bounds__(LBVH_THREADS)
hierarchy_kernel(const uint64_t* __restrict__ keys, const FrameState* __restrict__ st, int4* __restrict__ ranges, int wait_at_start) {
  if (wait_at_start) pdl_wait();
  pdl_trigger();
  const int n = (int)st->n;
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n - 1; i += gridDim.x * blockDim.x) {
    int first, gamma, last;
    karras_node(keys, n, i, first, gamma, last);
    ranges[i] = make_int4(first, gamma, last, 0);
  }
  if (!wait_at_start) pdl_wait();
}

__global__ void __launch_bounds__(LBVH_THREADS)
boxes_kernel(const int4* __restrict__ ranges, const float4* __restrict__ sphere, const float4* __restrict__ pyr,
             FrameState* st, Node* __restrict__ nodes) {
  pdl_wait();
  pdl_trigger();
  const int n = (int)st->n;
  if (n == 1 && blockIdx.x == 0 && threadIdx.x == 0) {  // the single leaf is the root
    float lo[3], hi[3];
    box_of_sphere(sphere[0], lo, hi);
#pragma unroll
    for (int a = 0; a < 3; ++a) { st->root_lo[a] = lo[a]; st->root_hi[a] = hi[a]; }
  }
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n - 1; i += gridDim.x * blockDim.x) {
    const int4 r = __ldg(ranges + i);
    write_node(sphere, pyr, st, nodes, i, r.x, r.y, r.z);
  }
}

// ===================================================================== tiled tree (default)
// splats_set_option(SPLATS_OPT_REFIT, SPLATS_REFIT_TILED): a4 and a5 in one pass over the sorted
// leaves, two launches.
//
// The radix tree over the sorted (key, position) pairs is the Cartesian tree of the adjacent
// common-prefix lengths d[g] = delta(g, g + 1): the internal node that splits between g and g + 1
// covers the leaves (p, q] where p (q) is the nearest position to the left (right) of g with a
// smaller d -- inside a node's range every other adjacent delta is larger than the one at its
// split, and the deltas just outside are smaller.  In Karras' numbering that node is `q` when it
// is a left child (d[q] > d[p]: the parent splits at q) and `p + 1` when it is a right child.
//
// tree_tile_kernel: one block per TT_LEAVES consecutive sorted leaves.  It gathers the splats
// into sorted order (as leaf_pyramid_kernel), keeps *all* levels of the tile's box pyramid and
// a min pyramid over the tile's deltas (one byte each: delta + 1 <= 96, 0 = "beyond the array")
// in shared memory, finds p and q of every split of the tile by a nearest-smaller-value search
// on the byte pyramid, and -- when both lie inside the tile, which is the case for all but the
// strict prefix / suffix minima of the tile's deltas (<= 2 x 97 nodes) -- takes both child boxes
// as range queries on the shared-memory box pyramid and writes the finished 64-byte node record.
// The other nodes go to a queue with what is known about them.
// tree_spine_kernel: finishes the queued nodes: missing range ends by galloping + 4-ary search
// on the sorted keys, boxes by range queries on the global pyramid (levels >= 1, written by the
// tile kernel; its top levels by the last block to finish).
// Same tree, same numbering, same boxes as the other two modes, bit for bit.
constexpr int TT_LOG = 10;
constexpr int TT_LEAVES = 1 << TT_LOG;
constexpr int TT_THREADS = 256;
constexpr int TT_PER = TT_LEAVES / TT_THREADS;
constexpr int TT_QMAX = 200;   // >= 2 x 97: strict prefix + suffix minima of byte-sized deltas
static_assert(TT_LOG == PYR_LOCAL, "the tile kernel writes the same global pyramid levels as leaf_pyramid_kernel");

__host__ __device__ __forceinline__ constexpr int tt_off(int k) { return 2 * TT_LEAVES - ((2 * TT_LEAVES) >> k); }

struct TileSmem {
  float box[6][2 * TT_LEAVES];   // level k (entries of 2^k leaves) at tt_off(k)
  uint8_t d[2 * TT_LEAVES];      // delta + 1 of the pair (l, l + 1), min pyramid at the same offsets
  int4 q[TT_QMAX];               // queued nodes: (split, first or -1, last or -1, 0)
  uint32_t qn, qbase;
  uint32_t dleft;                // delta + 1 of the pair (base - 1, base); 0 at the start of the array
  int last;
};

// first position q in [s, TT_LEAVES) with d[q] < v (level-0 positions), TT_LEAVES if there is none
__device__ __forceinline__ int nsv_right(const uint8_t* __restrict__ d, int s, uint32_t v) {
  int i = s, k = 0;
  while (true) {
    if ((i << k) >= TT_LEAVES) return TT_LEAVES;
    if (d[tt_off(k) + i] < v) break;
    ++i;                                        // everything in [s, i << k) is >= v
    const int up = min(__ffs(i) - 1, TT_LOG - k);   // the same position seen from a coarser level
    i >>= up;
    k += up;
  }
  while (k > 0) {
    --k;
    i <<= 1;
    if (d[tt_off(k) + i] >= v) ++i;
  }
  return i;
}
// last position p in [0, s] with d[p] < v, -1 if there is none
__device__ __forceinline__ int nsv_left(const uint8_t* __restrict__ d, int s, uint32_t v) {
  int i = s, k = 0;
  while (true) {
    if (i < 0) return -1;
    if (d[tt_off(k) + i] < v) break;
    --i;                                        // everything in ((i + 1) << k, s] is >= v
    if (i < 0) return -1;
    const int up = min(__ffs(i + 1) - 1, TT_LOG - k);   // trailing ones: blocks that end at the same position
    i >>= up;
    k += up;
  }
  while (k > 0) {
    --k;
    i = 2 * i + 1;
    if (d[tt_off(k) + i] >= v) --i;
  }
  return i;
}

// box of the tile-local leaves [l, r), l < r, from the shared-memory pyramid
__device__ __forceinline__ void range_box_tile(const float (*__restrict__ box)[2 * TT_LEAVES], int l, int r, float lo[3], float hi[3]) {
  const float INF = __int_as_float(0x7f800000);
#pragma unroll
  for (int a = 0; a < 3; ++a) { lo[a] = INF; hi[a] = -INF; }
  int off = 0, width = TT_LEAVES;
  while (l < r) {
    if (l & 1) {
#pragma unroll
      for (int a = 0; a < 3; ++a) { lo[a] = fminf(lo[a], box[a][off + l]); hi[a] = fmaxf(hi[a], box[3 + a][off + l]); }
      ++l;
    }
    if (r & 1) {
      --r;
#pragma unroll
      for (int a = 0; a < 3; ++a) { lo[a] = fminf(lo[a], box[a][off + r]); hi[a] = fmaxf(hi[a], box[3 + a][off + r]); }
    }
    l >>= 1;
    r >>= 1;
    off += width;
    width >>= 1;
  }
}

__device__ __forceinline__ void store_node(Node* __restrict__ nodes, int idx, const float llo[3], const float lhi[3],
                                           const float rlo[3], const float rhi[3], int first, int gamma, int last) {
  const int cnt_l = gamma - first + 1, cnt_r = last - gamma;
  const int left = cnt_l <= LEAF_MAX ? (int)leaf_range_code((uint32_t)first, (uint32_t)cnt_l) : gamma;
  const int right = cnt_r <= LEAF_MAX ? (int)leaf_range_code((uint32_t)gamma + 1u, (uint32_t)cnt_r) : gamma + 1;
  float4* rec = reinterpret_cast<float4*>(nodes + idx);
  rec[0] = make_float4(llo[0], llo[1], llo[2], lhi[0]);
  rec[1] = make_float4(lhi[1], lhi[2], rlo[0], rlo[1]);
  rec[2] = make_float4(rlo[2], rhi[0], rhi[1], rhi[2]);
  rec[3] = make_float4(__int_as_float(left), __int_as_float(right), 0.0f, 0.0f);
}

struct Box6 { float v[6]; };
__device__ __forceinline__ Box6 box_merge(const Box6& a, const Box6& b) {
  Box6 r;
#pragma unroll
  for (int k = 0; k < 3; ++k) { r.v[k] = fminf(a.v[k], b.v[k]); r.v[3 + k] = fmaxf(a.v[3 + k], b.v[3 + k]); }
  return r;
}

// Levels above TT_LOG of the global pyramid, by the last block of tree_tile_kernel to finish:
// five levels per round trip (a warp loads 32 consecutive entries and merges them with shuffles).
__device__ __forceinline__ void pyramid_top(float4* pyr, uint32_t cnt_prev, int k_prev) {
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  constexpr int NWARPS = TT_THREADS / 32;
  const float INF = __int_as_float(0x7f800000);
  while (cnt_prev > 1) {
    const float4* src = pyr + 2 * (size_t)c_pyr.off[k_prev];
    const uint32_t chunks = (cnt_prev + 31) >> 5;
    for (uint32_t c = warp; c < chunks; c += NWARPS) {
      const uint32_t j = c * 32 + lane;
      Box6 b;
      if (j < cnt_prev) {
        const float4 lo = __ldcg(src + 2 * (size_t)j), hi = __ldcg(src + 2 * (size_t)j + 1);
        b.v[0] = lo.x; b.v[1] = lo.y; b.v[2] = lo.z; b.v[3] = hi.x; b.v[4] = hi.y; b.v[5] = hi.z;
      } else {
#pragma unroll
        for (int a = 0; a < 3; ++a) { b.v[a] = INF; b.v[3 + a] = -INF; }
      }
#pragma unroll
      for (int s = 1; s <= 5; ++s) {
        Box6 o;
#pragma unroll
        for (int a = 0; a < 6; ++a) o.v[a] = __shfl_down_sync(0xffffffffu, b.v[a], 1 << (s - 1));
        b = box_merge(b, o);
        const uint32_t cnt = (cnt_prev + (1u << s) - 1) >> s;
        if ((lane & ((1 << s) - 1)) == 0 && (j >> s) < cnt && k_prev + s <= PYR_MAX_LEVELS) {
          float4* e = pyr + 2 * ((size_t)c_pyr.off[k_prev + s] + (j >> s));
          __stcg(e, make_float4(b.v[0], b.v[1], b.v[2], 0.0f));
          __stcg(e + 1, make_float4(b.v[3], b.v[4], b.v[5], 0.0f));
        }
      }
    }
    __syncthreads();
    cnt_prev = (cnt_prev + 31) >> 5;
    k_prev += 5;
  }
}

template <class Gather>
__global__ void __launch_bounds__(TT_THREADS)
tree_tile_kernel(const uint64_t* __restrict__ keys, const uint32_t* __restrict__ perm, const Gather src, FrameState* st,
                 float4* __restrict__ sphere, float4* __restrict__ rgba, uint32_t* __restrict__ ids_out, float4* pyr,
                 Node* __restrict__ nodes, int4* __restrict__ queue) {
  pdl_wait();
  pdl_trigger();
  extern __shared__ __align__(16) unsigned char tt_smem_raw[];
  TileSmem& s = *reinterpret_cast<TileSmem*>(tt_smem_raw);
  const int n = (int)st->n;
  const int nblocks = (n + TT_LEAVES - 1) / TT_LEAVES;
  if ((int)blockIdx.x >= nblocks) return;
  const int tid = threadIdx.x;
  const int base = blockIdx.x * TT_LEAVES;
  const float INF = __int_as_float(0x7f800000);

  // ---- deltas of the adjacent pairs (l, l + 1) of the tile, + 1; 0 beyond the array
  if (tid == 0) {
    s.qn = 0;
    uint32_t dl = 0;
    if (base > 0) {
      const uint64_t x = __ldg(keys + base - 1) ^ __ldg(keys + base);
      dl = 1u + (x ? (uint32_t)__clzll((long long)x) : 64u + (uint32_t)__clz((base - 1) ^ base));
    }
    s.dleft = dl;
  }
  uint32_t id[TT_PER];
#pragma unroll
  for (int j = 0; j < TT_PER; ++j) {
    const int i = base + tid + j * TT_THREADS;
    id[j] = i < n ? __ldg(perm + i) : 0u;
  }
#pragma unroll
  for (int j = 0; j < TT_PER; ++j) {
    const int l = tid + j * TT_THREADS, i = base + l;
    uint32_t dv = 0;
    if (i + 1 < n) {
      const uint64_t x = __ldg(keys + i) ^ __ldg(keys + i + 1);
      dv = 1u + (x ? (uint32_t)__clzll((long long)x) : 64u + (uint32_t)__clz(i ^ (i + 1)));
    }
    s.d[l] = (uint8_t)dv;
  }
  // ---- gather the splats of the tile into sorted order; leaf boxes -> level 0
#pragma unroll
  for (int j = 0; j < TT_PER; ++j) {
    const int l = tid + j * TT_THREADS, i = base + l;
    float lo[3] = {INF, INF, INF}, hi[3] = {-INF, -INF, -INF};
    if (i < n) {
      float4 sp, col;
      src.get(id[j], sp, col);
      sphere[i] = sp;
      rgba[i] = col;
      ids_out[i] = id[j];   // the BVH keeps its own copy: the sort buffers belong to the next build
      box_of_sphere(sp, lo, hi);
    }
#pragma unroll
    for (int a = 0; a < 3; ++a) { s.box[a][l] = lo[a]; s.box[3 + a][l] = hi[a]; }
  }
  if (n == 1 && tid == 0) {   // the single leaf is the root
#pragma unroll
    for (int a = 0; a < 3; ++a) { st->root_lo[a] = s.box[a][0]; st->root_hi[a] = s.box[3 + a][0]; }
  }
  __syncthreads();

  // ---- levels 1..TT_LOG of both pyramids (all levels stay in shared memory); the box levels
  // also go to the global pyramid for the queued nodes
#pragma unroll
  for (int k = 1; k <= TT_LOG; ++k) {
    const int cnt = TT_LEAVES >> k, o0 = tt_off(k - 1), o1 = tt_off(k);
    for (int j = tid; j < cnt; j += TT_THREADS) {
      float v[6];
#pragma unroll
      for (int a = 0; a < 3; ++a) {
        v[a] = fminf(s.box[a][o0 + 2 * j], s.box[a][o0 + 2 * j + 1]);
        v[3 + a] = fmaxf(s.box[3 + a][o0 + 2 * j], s.box[3 + a][o0 + 2 * j + 1]);
      }
#pragma unroll
      for (int a = 0; a < 6; ++a) s.box[a][o1 + j] = v[a];
      s.d[o1 + j] = min(s.d[o0 + 2 * j], s.d[o0 + 2 * j + 1]);
      if (base + (j << k) < n) {
        float4* e = pyr + 2 * ((size_t)c_pyr.off[k] + (base >> k) + j);
        __stcg(e, make_float4(v[0], v[1], v[2], 0.0f));
        __stcg(e + 1, make_float4(v[3], v[4], v[5], 0.0f));
      }
    }
    __syncthreads();
  }

  // ---- the nodes whose split lies in this tile
  const uint32_t dleft = s.dleft;
#pragma unroll 1
  for (int j = 0; j < TT_PER; ++j) {
    const int l = tid + j * TT_THREADS, g = base + l;
    if (g + 1 >= n) continue;
    const uint32_t v = s.d[l];
    const int q = nsv_right(s.d, l + 1, v);
    int p = l > 0 ? nsv_left(s.d, l - 1, v) : -1;
    bool open_l = false;
    if (p < 0) {                       // nothing smaller inside the tile: the pair (base - 1, base)?
      if (dleft < v) p = -1; else open_l = true;
    }
    const bool open_r = q >= TT_LEAVES;
    if (open_l || open_r) {
      const uint32_t slot = atomicAdd(&s.qn, 1u);
      s.q[slot] = make_int4(g, open_l ? -1 : base + p + 1, open_r ? -1 : base + q, 0);
      continue;
    }
    const int first = base + p + 1, last = base + q;
    const uint32_t dl = p < 0 ? dleft : s.d[p], dr = s.d[q];
    const int idx = dr > dl ? last : first;
    float llo[3], lhi[3], rlo[3], rhi[3];
    range_box_tile(s.box, p + 1, l + 1, llo, lhi);
    range_box_tile(s.box, l + 1, q + 1, rlo, rhi);
    store_node(nodes, idx, llo, lhi, rlo, rhi, first, g, last);
    if (idx == 0) {
#pragma unroll
      for (int a = 0; a < 3; ++a) { st->root_lo[a] = fminf(llo[a], rlo[a]); st->root_hi[a] = fmaxf(lhi[a], rhi[a]); }
    }
  }
  __syncthreads();
  const uint32_t qn = s.qn;
  if (qn) {
    if (tid == 0) s.qbase = atomicAdd(&st->spine_n, qn);
    __syncthreads();
    for (uint32_t e = tid; e < qn; e += TT_THREADS) queue[s.qbase + e] = s.q[e];
  }
  if (nblocks == 1) return;

  // ---- the last block to finish builds the levels above TT_LOG
  __threadfence();
  if (tid == 0) s.last = atomicAdd(&st->pyr_done, 1u) == (uint32_t)nblocks - 1u;
  __syncthreads();
  if (!s.last) return;
  __threadfence();
  pyramid_top(pyr, (uint32_t)nblocks, TT_LOG);
}

// Largest distance x >= x0 (in direction dir from g) with delta(g, g + x dir) >= dref, given that
// it holds at x0: gallop (x16 per round, four probes) then 4-ary descent.
__device__ __forceinline__ int spine_extend(const uint64_t* __restrict__ keys, int n, int g, uint64_t kg, int dir, int dref, int x0) {
  int lb = x0 > 0 ? x0 : 1, base = x0;
  // invariant: holds at `base`; find a power-of-two step that fails
  int step = 1;
  while (step < lb) step <<= 1;
  while (true) {
    const int c = (int)(delta(keys, n, g, kg, g + (base + step) * dir) >= dref) + (int)(delta(keys, n, g, kg, g + (base + 2 * step) * dir) >= dref) +
                  (int)(delta(keys, n, g, kg, g + (base + 4 * step) * dir) >= dref) + (int)(delta(keys, n, g, kg, g + (base + 8 * step) * dir) >= dref);
    // the predicate is monotone in the distance: c probes hold, the next one fails
    if (c == 0) break;
    base += step << (c - 1);
    if (c < 4) { step <<= (c - 1); break; }
    step <<= 4;
  }
  // holds at base, fails at base + step
  int width = step;
  while (width >= 4) {
    const int qd = width >> 2;
    const int c = (int)(delta(keys, n, g, kg, g + (base + qd) * dir) >= dref) + (int)(delta(keys, n, g, kg, g + (base + 2 * qd) * dir) >= dref) +
                  (int)(delta(keys, n, g, kg, g + (base + 3 * qd) * dir) >= dref);
    base += c * qd;
    width = qd;
  }
  if (width == 2 && delta(keys, n, g, kg, g + (base + 1) * dir) >= dref) base += 1;
  return base;
}

__global__ void __launch_bounds__(LBVH_THREADS)
tree_spine_kernel(const uint64_t* __restrict__ keys, FrameState* st, const int4* __restrict__ queue,
                  const float4* __restrict__ sphere, const float4* __restrict__ pyr, Node* __restrict__ nodes) {
  pdl_wait();
  pdl_trigger();
  const int n = (int)st->n;
  const int qn = (int)st->spine_n;
  for (int e = blockIdx.x * blockDim.x + threadIdx.x; e < qn; e += gridDim.x * blockDim.x) {
    const int4 ent = __ldg(queue + e);
    const int g = ent.x;
    const uint64_t kg = __ldg(keys + g);
    const int dnode = delta(keys, n, g, kg, g + 1);
    const int tile_lo = g & ~(TT_LEAVES - 1), tile_hi = min(tile_lo + TT_LEAVES - 1, n - 1);
    // an open end lies beyond the tile: start the search at the tile's edge
    const int first = ent.y >= 0 ? ent.y : g - spine_extend(keys, n, g, kg, -1, dnode, g - tile_lo);
    const int last = ent.z >= 0 ? ent.z : g + spine_extend(keys, n, g, kg, +1, dnode, tile_hi - g);
    const int dl = first > 0 ? delta(keys, n, first - 1, __ldg(keys + first - 1), first) : -1;
    const int dr = last < n - 1 ? delta(keys, n, last, __ldg(keys + last), last + 1) : -1;
    const int idx = dr > dl ? last : first;
    write_node(sphere, pyr, st, nodes, idx, first, g, last);
  }
}

// Canonical export for the bit-exact acceptance checks (include/splats.h, splats_export).
// Parent links are not part of the traversal structure: they are derived here from the
// child links (parents[] must be pre-filled with -1 by the caller; the root keeps it).
__global__ void __launch_bounds__(LBVH_THREADS)
export_kernel(const Node* __restrict__ nodes, const float4* __restrict__ sphere,
              const FrameState* __restrict__ st, int* __restrict__ children, int* __restrict__ parents,
              float* __restrict__ aabbs) {
  const int n = (int)st->n;
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
    const int leaf_id = n - 1 + i;
    if (aabbs) {
      float* bx = aabbs + 6 * (size_t)leaf_id;
      box_of_sphere(sphere[i], bx, bx + 3);
    }
    if (i < n - 1) {
      const Node nd = nodes[i];
      // canonical Karras links from the traversal links (common.cuh, Node)
      const uint32_t l = (uint32_t)nd.left, r = (uint32_t)nd.right;
      int cl = nd.left, cr = nd.right;
      if (nd.left < 0) {
        const int f = (int)leaf_range_first(l), c = (int)leaf_range_count(l);
        cl = c == 1 ? n - 1 + f : f + c - 1;
      }
      if (nd.right < 0) {
        const int f = (int)leaf_range_first(r), c = (int)leaf_range_count(r);
        cr = c == 1 ? n - 1 + f : f;
      }
      if (children) {
        children[2 * i] = cl;
        children[2 * i + 1] = cr;
      }
      if (parents) {
        parents[cl] = i;
        parents[cr] = i;
      }
      if (aabbs) {
        float* bx = aabbs + 6 * (size_t)i;
#pragma unroll
        for (int a = 0; a < 3; ++a) {
          bx[a] = fminf(nd.b[a], nd.b[6 + a]);
          bx[3 + a] = fmaxf(nd.b[3 + a], nd.b[9 + a]);
        }
      }
    }
  }
}

}  // namespace sw
