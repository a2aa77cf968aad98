// lbvh.cuh -- steps a4 (Karras-style hierarchy emission) and a5 (bottom-up refit with atomic
// arrival counters) of SURVEY.md sec. 8(a), plus the canonical export used by the parity
// tests.  "build a bounding volume hierarchy ... using the LBVH algorithm".
#pragma once
#include "common.cuh"

namespace sw {

constexpr int LBVH_THREADS = 256;

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
__global__ void __launch_bounds__(LBVH_THREADS)
emit_kernel(const uint64_t* __restrict__ keys, const uint32_t* __restrict__ perm,
            const float* __restrict__ depth, const float4* __restrict__ color, DevCamera cam, float k_r,
            const FrameState* __restrict__ st, float4* __restrict__ sphere, float4* __restrict__ rgba,
            Node* __restrict__ nodes, int* __restrict__ leaf_parent) {
  const int n = (int)st->n;
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
    // ---- (a) gather
    const uint32_t id = __ldg(perm + i);
    const int y = (int)(id / (uint32_t)cam.W), x = (int)(id - (uint32_t)y * (uint32_t)cam.W);
    const float t = __ldg(depth + id);
    float p[3], len;
    splat_centre(cam, x, y, t, p, len);
    const float z = div_(t, len);
    sphere[i] = make_float4(p[0], p[1], p[2], mul_(k_r, z));
    rgba[i] = __ldg(color + id);
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

// Canonical export for the bit-exact acceptance checks (include/splats.h, splats_export).
__global__ void __launch_bounds__(LBVH_THREADS)
export_kernel(const Node* __restrict__ nodes, const int* __restrict__ leaf_parent,
              const float4* __restrict__ sphere, const FrameState* __restrict__ st,
              int* __restrict__ children, int* __restrict__ parents, float* __restrict__ aabbs) {
  const int n = (int)st->n;
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
    const int leaf_id = n - 1 + i;
    if (parents) parents[leaf_id] = leaf_parent[i] < 0 ? -1 : (leaf_parent[i] >> 1);
    if (aabbs) {
      const float4 sp = sphere[i];
      float* bx = aabbs + 6 * (size_t)leaf_id;
      bx[0] = sub_(sp.x, sp.w); bx[1] = sub_(sp.y, sp.w); bx[2] = sub_(sp.z, sp.w);
      bx[3] = add_(sp.x, sp.w); bx[4] = add_(sp.y, sp.w); bx[5] = add_(sp.z, sp.w);
    }
    if (i < n - 1) {
      const Node nd = nodes[i];
      if (children) {
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
        children[2 * i] = cl;
        children[2 * i + 1] = cr;
      }
      if (parents) parents[i] = nd.parent < 0 ? -1 : (nd.parent >> 1);
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
