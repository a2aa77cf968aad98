// lbvh.cuh -- steps a4 (Karras-style hierarchy emission) and a5 (bottom-up refit with atomic
// arrival counters) of SURVEY.md sec. 8(a), plus the canonical export used by the parity
// tests.  "build a bounding volume hierarchy ... using the LBVH algorithm".
#pragma once
#include "common.cuh"

namespace sw {

constexpr int LBVH_THREADS = 256;

// Splat `id` (= source pixel index, or position in a received sample buffer) as sphere + colour.
// FrameGather reads the splat that bounds_kernel stored for that pixel (Eq. 1; radius
// per RadiusParams: evaluated once per frame) and copies the colour ("no shading
// other than the constant sample color"); PackedGather decodes the
// 64-bit sample and the RGBA8 colour.
struct FrameGather {
  const float4* __restrict__ sphere_px;   // splat of every valid pixel, written by bounds_kernel (Eq. 1 once)
  const float4* __restrict__ color;
  __device__ __forceinline__ void get(uint32_t id, float4& sp, float4& col) const {
    sp = __ldg(sphere_px + id);
    col = __ldg(color + id);
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
// Invariant behind wait_at_start = 0 (and behind renders / bounds_kernel that skip the wait): the kernel only reads
// what a grid BEFORE its predecessor in the stream produced (here: the sorted keys, written by onesweep_kernel; the
// predecessor is leaf_pyramid_kernel).  That grid has retired: every block of the predecessor passed its own
// griddepcontrol.wait, i.e. saw that grid complete and flushed, before this kernel could be released.
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

// Canonical export for the bit-exact acceptance checks (include/splats.h, splats_export).
// The other two refit modes (SPLATS_REFIT_PYRAMID, SPLATS_REFIT_ATOMIC) produce exact 64-byte
// records; the traversal reads the 32-byte quantised ones (common.cuh, QNode): one more pass.
__global__ void __launch_bounds__(LBVH_THREADS)
quantise_nodes_kernel(const Node* __restrict__ nodes, const FrameState* __restrict__ st, QNode* __restrict__ qnodes) {
  pdl_wait();
  pdl_trigger();
  const int n = (int)st->n;
  const QFrame q = load_qframe(st);
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n - 1; i += gridDim.x * blockDim.x) {
    const float4* rec = reinterpret_cast<const float4*>(nodes + i);
    const float4 a = __ldcg(rec), b = __ldcg(rec + 1), c = __ldcg(rec + 2), d = __ldcg(rec + 3);
    const float L[6] = {a.x, a.y, a.z, a.w, b.x, b.y}, R[6] = {b.z, b.w, c.x, c.y, c.z, c.w};
    store_qnode(qnodes + i, L, R, __float_as_int(d.x), __float_as_int(d.y), q);
  }
}

// The sorted keys are kept as code << 1 (build_kernels.cuh): give the codes back.
__global__ void __launch_bounds__(LBVH_THREADS)
export_keys_kernel(const uint64_t* __restrict__ keys, const FrameState* __restrict__ st, uint64_t* __restrict__ out) {
  const int n = (int)st->n;
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) out[i] = keys[i] >> 1;
}

// Parent links are not part of the traversal structure: they are derived here from the
// child links (parents[] must be pre-filled with -1 by the caller; the root keeps it).
// Topology comes from the traversal records; the exact boxes from the 64-byte records, which
// exist only when the build wrote them (`nodes` may be null: then aabbs must be null too).
__global__ void __launch_bounds__(LBVH_THREADS)
export_kernel(const QNode* __restrict__ qnodes, const Node* __restrict__ nodes, const float4* __restrict__ sphere,
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
      // canonical Karras links from the traversal links (common.cuh, Node)
      const uint32_t l = qnodes[i].w[6], r = qnodes[i].w[7];
      int cl = (int)l, cr = (int)r;
      if (cl < 0) {
        const int f = (int)leaf_range_first(l), c = (int)leaf_range_count(l);
        cl = c == 1 ? n - 1 + f : f + c - 1;
      }
      if (cr < 0) {
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
        const Node nd = nodes[i];
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
