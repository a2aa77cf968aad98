// tree_tile.cuh -- steps a4 + a5 of SURVEY.md sec. 8(a) in one pass over the sorted leaves
// (splats_set_option(SPLATS_OPT_REFIT, SPLATS_REFIT_TILED), the default): "build a bounding
// volume hierarchy ... using the LBVH algorithm".
//
// The radix tree over the sorted (key, position) pairs is the Cartesian tree of the adjacent
// common-prefix lengths d[g] = delta(g, g + 1): the internal node that splits between g and g + 1
// covers the leaves (p, q] where p (q) is the nearest position to the left (right) of g with a
// smaller d -- inside a node's range every other adjacent delta is larger than the one at its
// split, and the two just outside are smaller.  The parent of a subtree over (p, q] is therefore
// the node that splits at q if d[q] > d[p] (the subtree is its left child) and the one that splits
// at p otherwise, and in Karras' numbering the node over (p, q] is `q` in the first case and
// `p + 1` in the second.
//
// Boxes are carried as QBox (common.cuh): six 16-bit codes in three words whose union is three packed
// minima.  Quantisation is monotone, so the union of quantised boxes is the quantised exact union:
// the records equal quantise(exact child boxes) (S13 of DESIGN.md) bit for bit, and no float box is
// ever formed after the leaves.  (The exact float32 records of SPLATS_OPT_EXACT_NODES come from the
// pyramid refit, lbvh.cuh, run after this one.)
//
// tree_tile_kernel: one block per TT_LEAVES consecutive sorted leaves.  It gathers the splats into
// sorted order, writes the levels >= PYR_BASE of the global box pyramid (registers + shuffles),
// and builds every subtree that lies inside the tile bottom-up in shared memory: a finished
// subtree stores its box and the far end of its range in its parent's slot and sets its arrival
// bit; the second arrival appends the parent to a work list; one round per tree level, each round
// dense over the work list (no lane waits for a long node).  After the rounds every node whose
// children both arrived is written out as its 32-byte record.  The nodes with a missing child -- their range
// crosses a tile edge; they are strict prefix / suffix minima of the tile's deltas, <= 2 x 97 per
// tile -- are queued with what is known about them.  The block also writes, for every threshold
// v, the position of the first / last split of the tile with d < v.
// tree_spine_kernel: finishes the queued nodes, one warp each: the missing range end is the first
// (last) split with a smaller delta in the nearest tile that has one (a search over one byte per
// tile in shared memory, then one table look-up); the two child boxes are range queries on the
// global pyramid whose <= 76 independent pieces are spread over the lanes (one round trip).
// Same tree, same numbering, same boxes as the other two modes, bit for bit.
#pragma once
#include "lbvh.cuh"

namespace sw {

#ifndef SPLATS_TT_LOG
#define SPLATS_TT_LOG 10
#endif
constexpr int TT_LOG = SPLATS_TT_LOG;
constexpr int TT_LEAVES = 1 << TT_LOG;
constexpr int TT_THREADS = TT_LEAVES / 4;    // a thread owns four consecutive leaves
constexpr int TT_WARPS = TT_THREADS / 32;
constexpr int TT_QMAX = 200;    // >= 2 x 97: strict prefix + suffix minima of byte-sized deltas
constexpr int TT_VMAX = 97;     // delta + 1 lies in [0, 96]; 0 = "beyond the array"
constexpr int TT_VPAD = 100;    // table stride
#ifndef SPLATS_TT_CLIMB
#define SPLATS_TT_CLIMB 64
#endif
constexpr int TT_CLIMB = SPLATS_TT_CLIMB;    // work lists up to this length are finished by climbing threads instead of block-wide rounds
constexpr int PYR_BASE = 3;     // lowest level of the global pyramid that the tiled mode writes and reads
static_assert(TT_LOG >= 7 && TT_LOG <= 12, "tile of 128 .. 4096 leaves");

struct TileSmem {
  uint32_t cbox[2][3][TT_LEAVES];   // [side][word][split]: child boxes (QBox: six 16-bit codes) of the node that splits at l.
                                    // cbox[0] doubles as the staging of the leaf boxes before round 0.
  int16_t cend[2][TT_LEAVES];    // far end of each child's range: tile-local p (left child) or q (right child)
  uint32_t arrived[TT_LEAVES / 4];   // one byte per split: bit 0 left child stored, bit 1 right child stored
  uint16_t wl[TT_LEAVES];        // finished nodes in completion order (each node enters once)
  uint8_t d[TT_LEAVES];          // delta + 1 of the pair (l, l + 1); 0 beyond the array
  uint32_t pos_first[TT_VPAD];   // first / last split of the tile with d == u
  int32_t pos_last[TT_VPAD];
  uint32_t top[3][TT_WARPS];     // the warps' level-7 entries
  uint32_t wmin[TT_WARPS];       // the warps' smallest delta + 1
  int4 q[TT_QMAX];               // queued nodes: (split, first or -1, last or -1, delta + 1)
  uint32_t cnt[3];               // lengths of the work lists of rounds r % 3
  uint32_t qn, qbase;
  uint32_t dleft;                // delta + 1 of the pair (base - 1, base); 0 at the start of the array
  int last;
};

// Slot of split l in cbox / cend during the rounds: XOR swizzle, so that the power-of-two strides
// the work lists start with (4 leaves per thread, every other split finished) hit 32 different banks.
__device__ __forceinline__ int tt_slot(int l) { return l ^ ((l >> 5) & 31); }

// The global pyramid of the tiled mode holds QBox entries (16 bytes each, word 3 unused) in the buffer the
// pyramid mode uses for its float boxes; same level offsets (c_pyr, in entries).
__device__ __forceinline__ void pyr_store(uint4* pyr, int level, uint32_t index, const QBox& b) {
  __stcg(pyr + (size_t)c_pyr.off[level] + index, make_uint4(b.w[0], b.w[1], b.w[2], 0u));
}

// Levels above `k_prev` of the global pyramid, by the last block of tree_tile_kernel to finish:
// five levels per round trip (a warp loads 32 consecutive entries and merges them with shuffles).
__device__ __forceinline__ void pyramid_top(uint4* pyr, uint32_t cnt_prev, int k_prev) {
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  while (cnt_prev > 1) {
    const uint4* src = pyr + (size_t)c_pyr.off[k_prev];
    const uint32_t chunks = (cnt_prev + 31) >> 5;
    for (uint32_t c = warp; c < chunks; c += TT_WARPS) {
      const uint32_t j = c * 32 + lane;
      QBox b;
      b.init();
      if (j < cnt_prev) {
        const uint4 e = __ldcg(src + j);
        b.w[0] = e.x; b.w[1] = e.y; b.w[2] = e.z;
      }
#pragma unroll
      for (int s = 1; s <= 5; ++s) {
        b.merge(b.shfl_down(1 << (s - 1)));
        const uint32_t cnt = (cnt_prev + (1u << s) - 1) >> s;
        if ((lane & ((1 << s) - 1)) == 0 && (j >> s) < cnt && k_prev + s <= PYR_MAX_LEVELS) pyr_store(pyr, k_prev + s, j >> s, b);
      }
    }
    __syncthreads();
    cnt_prev = (cnt_prev + 31) >> 5;
    k_prev += 5;
  }
}

// A finished subtree over the tile-local leaves (p, q] with box b reports to its parent: the node
// that splits at q when d[q] > d[p] (left child), else the one that splits at p (right child).
// Returns the parent's split if this was the second arrival (the parent is complete), -1 otherwise
// or when the parent lies in the tile to the left.  `is_last` = Karras: the subtree's own node
// index is its last leaf (it is a left child), else its first.
__device__ __forceinline__ int tile_report(TileSmem& s, int p, int q, const QBox& b, bool& is_last) {
  const uint32_t dl = p < 0 ? s.dleft : s.d[p], dr = s.d[q];
  is_last = dr > dl;
  int g, side, far;
  if (is_last) { g = q; side = 0; far = p; }
  else { if (p < 0) return -1; g = p; side = 1; far = q; }
  const int gs = tt_slot(g);
#pragma unroll
  for (int a = 0; a < 3; ++a) s.cbox[side][a][gs] = b.w[a];
  s.cend[side][gs] = (int16_t)far;
  __threadfence_block();   // the slot is written before the arrival bit is visible
  const int sh = 8 * (g & 3);
  const uint32_t old = atomicOr(&s.arrived[g >> 2], (1u << side) << sh);
  return ((old >> sh) & 3u) == (2u >> side) ? g : -1;   // the other bit was already set
}

template <class Gather>
#ifndef SPLATS_TT_BLOCKS
#define SPLATS_TT_BLOCKS 5   // resident blocks per SM the register allocation aims at (48 registers; 4 .. 6 measured)
#endif
__global__ void __launch_bounds__(TT_THREADS, SPLATS_TT_BLOCKS)
tree_tile_kernel(const uint64_t* __restrict__ keys, const uint32_t* __restrict__ perm, const Gather src, FrameState* st,
                 float4* __restrict__ sphere, float4* __restrict__ rgba, uint32_t* __restrict__ ids_out, uint4* pyr,
                 QNode* __restrict__ qnodes, int4* __restrict__ queue, uint8_t* __restrict__ tile_min,
                 uint16_t* __restrict__ tile_fb) {
  pdl_wait();
#if !SPLATS_LATE_TRIGGER
  pdl_trigger();
#endif
  extern __shared__ __align__(16) unsigned char tt_smem_raw[];
  TileSmem& s = *reinterpret_cast<TileSmem*>(tt_smem_raw);
  const int n = (int)st->n;
  const int nblocks = (n + TT_LEAVES - 1) / TT_LEAVES;
  if ((int)blockIdx.x >= nblocks) return;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int base = blockIdx.x * TT_LEAVES;
  const QFrame qf = load_qframe(st);

  // ---- (1) interleaved over the tile (coalesced): deltas of the adjacent pairs (l, l + 1), + 1;
  // gather of the splats into sorted order; leaf boxes -> staging
  if (tid == 0) {
    s.cnt[0] = 0; s.cnt[1] = 0; s.cnt[2] = 0;
    s.qn = 0;
    uint32_t dl = 0;
    if (base > 0) {
      const uint64_t x = __ldg(keys + base - 1) ^ __ldg(keys + base);
      dl = 1u + (x ? (uint32_t)__clzll((long long)x) : 64u + (uint32_t)__clz((base - 1) ^ base));
    }
    s.dleft = dl;
  }
  if (tid < TT_VPAD) { s.pos_first[tid] = TT_LEAVES; s.pos_last[tid] = -1; }
  s.arrived[tid] = 0u;
  uint32_t id[4];
#pragma unroll
  for (int j = 0; j < 4; ++j) {
    const int i = base + tid + j * TT_THREADS;
    id[j] = i < n ? __ldg(perm + i) : 0u;
  }
#pragma unroll
  for (int j = 0; j < 4; ++j) {
    const int l = tid + j * TT_THREADS, i = base + l;
    uint32_t dv = 0;
    if (i + 1 < n) {
      const uint64_t x = __ldg(keys + i) ^ __ldg(keys + i + 1);
      dv = 1u + (x ? (uint32_t)__clzll((long long)x) : 64u + (uint32_t)__clz(i ^ (i + 1)));
    }
    s.d[l] = (uint8_t)dv;
  }
#pragma unroll
  for (int j = 0; j < 4; ++j) {
    const int l = tid + j * TT_THREADS, i = base + l;
    QBox lb;
    lb.init();
    if (i < n) {
      float4 sp, col;
      src.get(id[j], sp, col);
      sphere[i] = sp;
      rgba[i] = col;
      ids_out[i] = id[j];   // the BVH keeps its own copy: the sort buffers belong to the next build
      lb = quant_sphere(sp, qf);
    }
#pragma unroll
    for (int a = 0; a < 3; ++a) s.cbox[0][a][l] = lb.w[a];
  }
  __syncthreads();

  // ---- (2) consecutive: thread t owns the leaves 4t .. 4t+3.  Leaf boxes into registers; global
  // pyramid levels PYR_BASE .. TT_LOG by shuffles (levels 1, 2 exist only in registers).
  QBox leaf[4];
  {
    uint4 c[3];
#pragma unroll
    for (int a = 0; a < 3; ++a) c[a] = *reinterpret_cast<const uint4*>(&s.cbox[0][a][4 * tid]);
#pragma unroll
    for (int a = 0; a < 3; ++a) { leaf[0].w[a] = c[a].x; leaf[1].w[a] = c[a].y; leaf[2].w[a] = c[a].z; leaf[3].w[a] = c[a].w; }
  }
  const int valid = min(TT_LEAVES, n - base);   // leaves of this tile = its splits, the last one of the array (d + 1 = 0) included
  // the tile's deltas: strict prefix / suffix minima (for the spine kernel's tables), smallest value
  uint32_t dk[4];
  {
    const uint32_t dword = *reinterpret_cast<const uint32_t*>(&s.d[4 * tid]);
#pragma unroll
    for (int k = 0; k < 4; ++k) dk[k] = 4 * tid + k < valid ? (dword >> (8 * k)) & 0xffu : 255u;
  }
  uint32_t pre = min(min(dk[0], dk[1]), min(dk[2], dk[3])), suf = pre;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const uint32_t a = __shfl_up_sync(0xffffffffu, pre, o), b = __shfl_down_sync(0xffffffffu, suf, o);
    if (lane >= o) pre = min(pre, a);
    if (lane + o < 32) suf = min(suf, b);
  }
  if (lane == 31) s.wmin[warp] = pre;
  uint32_t pre_ex = __shfl_up_sync(0xffffffffu, pre, 1), suf_ex = __shfl_down_sync(0xffffffffu, suf, 1);
  if (lane == 0) pre_ex = 255u;
  if (lane == 31) suf_ex = 255u;
  {
    QBox b = leaf[0];
    b.merge(leaf[1]); b.merge(leaf[2]); b.merge(leaf[3]);   // level 2 entry (base >> 2) + tid
#pragma unroll
    for (int sft = 1; sft <= 5; ++sft) {                        // levels 3 .. 7
      b.merge(b.shfl_down(1 << (sft - 1)));
      const int level = 2 + sft;
      if (level >= PYR_BASE && level <= TT_LOG && (lane & ((1 << sft) - 1)) == 0 && base + 4 * tid < n)
        pyr_store(pyr, level, (uint32_t)(base + 4 * tid) >> level, b);
    }
    if (TT_LOG > 7 && lane == 0) {
#pragma unroll
      for (int a = 0; a < 3; ++a) s.top[a][warp] = b.w[a];
    }
  }
  __syncthreads();   // every thread holds its leaf boxes: cbox[0] is free for the rounds below
  if (TT_LOG > 7 && warp == 0) {                                // levels 8 .. TT_LOG from the warps' entries
    QBox b;
    b.init();
    if (lane < TT_WARPS) {
#pragma unroll
      for (int a = 0; a < 3; ++a) b.w[a] = s.top[a][lane];
    }
#pragma unroll
    for (int sft = 1; sft <= TT_LOG - 7; ++sft) {
      b.merge(b.shfl_down(1 << (sft - 1)));
      if ((lane & ((1 << sft) - 1)) == 0 && lane < TT_WARPS && base + 128 * lane < n)
        pyr_store(pyr, 7 + sft, (uint32_t)(base + 128 * lane) >> (7 + sft), b);
    }
  }
  {   // strict prefix (suffix) minima of the tile's deltas: the only candidates for "first (last) split with d < v"
#pragma unroll
    for (int w = 0; w < TT_WARPS; ++w) {
      const uint32_t x = s.wmin[w];
      if (w < warp) pre_ex = min(pre_ex, x);
      if (w > warp) suf_ex = min(suf_ex, x);
    }
#pragma unroll
    for (int k = 0; k < 4; ++k)
      if (dk[k] < pre_ex) { s.pos_first[dk[k]] = 4 * tid + k; pre_ex = dk[k]; }
#pragma unroll
    for (int k = 3; k >= 0; --k)
      if (dk[k] < suf_ex) { s.pos_last[dk[k]] = 4 * tid + k; suf_ex = dk[k]; }
  }

  // ---- (3) round 0: the leaves report to their parents.  Finished nodes go to the work list; the
  // list of round r + 1 starts where that of round r ends, its length is counted in cnt[(r + 1) % 3]
  // (three rotating counters: one barrier per round is enough).
  auto append = [&](int g, uint32_t at, uint32_t* counter) {   // warp-aggregated push (g < 0: nothing); all 32 lanes call it
    const unsigned m = __ballot_sync(0xffffffffu, g >= 0);
    if (m) {
      const int leader = __ffs(m) - 1;
      uint32_t pos = 0;
      if (lane == leader) pos = atomicAdd(counter, (uint32_t)__popc(m));
      pos = __shfl_sync(0xffffffffu, pos, leader);
      if (g >= 0) s.wl[at + pos + __popc(m & ((1u << lane) - 1))] = (uint16_t)g;
    }
  };
  // a finished node reports upwards; returns the parent if that completed it.  (Its record is written
  // after the rounds, from the slots: nothing but the propagation is on the rounds' critical path.)
  auto finish = [&](int l) -> int {
    const int ls = tt_slot(l);
    const int p = s.cend[0][ls], q = s.cend[1][ls];
    QBox U, R;
#pragma unroll
    for (int a = 0; a < 3; ++a) { U.w[a] = s.cbox[0][a][ls]; R.w[a] = s.cbox[1][a][ls]; }
    U.merge(R);
    bool il;
    return tile_report(s, p, q, U, il);
  };
#pragma unroll
  for (int j = 0; j < 4; ++j) {
    const int i = 4 * tid + j;
    int g = -1;
    if (i < valid) {
      bool il;
      g = tile_report(s, i - 1, i, leaf[j], il);
    }
    append(g, 0u, &s.cnt[1]);
  }
  __syncthreads();

  // ---- dense rounds while the list is long: the nodes completed in the previous round are written
  // out and report upwards, one node per thread whatever its size
  uint32_t begin = 0;
  int r = 1;
  uint32_t len = s.cnt[1];
  while (len > TT_CLIMB) {
    if (tid == 0) s.cnt[(r + 2) % 3] = 0u;   // read in round r - 1, appended to in round r + 1
    uint32_t* next = &s.cnt[(r + 1) % 3];
    for (uint32_t e0 = 0; e0 < len; e0 += TT_THREADS) {
      const uint32_t e = e0 + tid;
      append(e < len ? finish(s.wl[begin + e]) : -1, begin + len, next);
    }
    __syncthreads();
    begin += len;
    ++r;
    len = s.cnt[r % 3];
  }
  // ---- the few nodes left climb on their own: no more barriers.  A subtree's stores are fenced
  // before its arrival bit is set (tile_report); whoever sets the second bit fences again and may
  // read both slots.
  if (tid < len) {
    int l = s.wl[begin + tid];
    while (l >= 0) {
      __threadfence_block();
      l = finish(l);
    }
  }
  // the last block to get here finishes the global pyramid at its end.  Only this thread's store of the tile's
  // top pyramid entry (phase 2) has to be visible to it, so only this thread fences, long after that store
  // (a fence by every thread at the end of the kernel waited for all of the block's stores: 10 % of the kernel)
  if (tid == 0 && nblocks > 1) {
    __threadfence();
    s.last = atomicAdd(&st->tile_done, 1u) == (uint32_t)nblocks - 1u;
  }
  __syncthreads();

  // ---- every split of the tile, dense: a complete node (both children arrived) is written out as its
  // traversal record (and, on request, the exact 64-byte record); an incomplete one is queued with
  // what is known
#pragma unroll 1
  for (int j = 0; j < 4; ++j) {
    const int l = tid + j * TT_THREADS, g = base + l;
    if (g + 1 >= n) continue;
    const uint32_t arr = (s.arrived[l >> 2] >> (8 * (l & 3))) & 3u;
    const int ls = tt_slot(l);
    if (arr != 3u) {
      const uint32_t slot = atomicAdd(&s.qn, 1u);
      s.q[slot] = make_int4(g, (arr & 1u) ? base + s.cend[0][ls] + 1 : -1, (arr & 2u) ? base + s.cend[1][ls] : -1, (int)s.d[l]);
      continue;
    }
    const int p = s.cend[0][ls], q = s.cend[1][ls];
    QBox L, R;
#pragma unroll
    for (int a = 0; a < 3; ++a) { L.w[a] = s.cbox[0][a][ls]; R.w[a] = s.cbox[1][a][ls]; }
    const uint32_t dl = p < 0 ? s.dleft : s.d[p], dr = s.d[q];
    const int first = base + p + 1, last = base + q;
    const int idx = dr > dl ? last : first;   // Karras: a left child is numbered by its last leaf, a right child by its first
    const int cnt_l = g - first + 1, cnt_r = last - g;
    const int left = cnt_l <= LEAF_MAX ? (int)leaf_range_code((uint32_t)first, (uint32_t)cnt_l) : g;
    const int right = cnt_r <= LEAF_MAX ? (int)leaf_range_code((uint32_t)g + 1u, (uint32_t)cnt_r) : g + 1;
    store_qnode(qnodes + idx, L, R, left, right);
  }
  __syncthreads();
  const uint32_t qn = s.qn;
  if (qn) {
    if (tid == 0) s.qbase = atomicAdd(&st->spine_n, qn);
    __syncthreads();
    for (uint32_t e = tid; e < qn; e += TT_THREADS) queue[s.qbase + e] = s.q[e];
  }
  // ---- tables for the spine kernel: tile_fb[v] = first split of the tile with d + 1 < v (TT_LEAVES: none),
  // tile_fb[TT_VPAD + v] = last one (0xffff: none); tile_min = smallest d + 1
  if (warp == 1 % TT_WARPS) {
    uint32_t f[4], fm = TT_LEAVES;
    int32_t g[4], gm = -1;
#pragma unroll
    for (int k = 0; k < 4; ++k) {   // lane holds u = 4 lane + k: exclusive running min / max over u
      const int u = 4 * lane + k;
      f[k] = fm;
      g[k] = gm;
      if (u < TT_VPAD) { fm = min(fm, s.pos_first[u]); gm = max(gm, s.pos_last[u]); }
    }
    uint32_t fi = fm;
    int32_t gi = gm;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {   // inclusive scan of the lane totals
      const uint32_t of = __shfl_up_sync(0xffffffffu, fi, o);
      const int32_t og = __shfl_up_sync(0xffffffffu, gi, o);
      if (lane >= o) { fi = min(fi, of); gi = max(gi, og); }
    }
    const uint32_t pf = __shfl_up_sync(0xffffffffu, fi, 1);
    const int32_t pg = __shfl_up_sync(0xffffffffu, gi, 1);
    uint16_t* fb = tile_fb + (size_t)blockIdx.x * (2 * TT_VPAD);
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      const int v = 4 * lane + k;
      if (v < TT_VPAD) {
        const uint32_t a = lane > 0 ? min(f[k], pf) : f[k];
        const int32_t b2 = lane > 0 ? max(g[k], pg) : g[k];
        fb[v] = (uint16_t)a;
        fb[TT_VPAD + v] = (uint16_t)(b2 < 0 ? 0xffff : b2);
      }
    }
  }
  if (tid == 0) {
    uint32_t m = 255u;
#pragma unroll
    for (int w = 0; w < TT_WARPS; ++w) m = min(m, s.wmin[w]);
    tile_min[blockIdx.x] = (uint8_t)m;
  }
  // ---- the last block builds the pyramid levels above TT_LOG
  if (nblocks == 1 || !s.last) return;
  __threadfence();
  pyramid_top(pyr, (uint32_t)nblocks, TT_LOG);
}

// ---- spine
// min pyramid over one byte per tile in shared memory: level k at off(k) = 2 NT - (2 NT >> k)
struct TileMins {
  const uint8_t* m;
  int nt, log;   // NT = 2^log entries at level 0
  __device__ __forceinline__ int off(int k) const { return 2 * nt - ((2 * nt) >> k); }
  // nearest tile t' >= s with m[t'] < v, nt if there is none
  __device__ __forceinline__ int right(int s, uint32_t v) const {
    int i = s, k = 0;
    while (true) {
      if ((i << k) >= nt) return nt;
      if (m[off(k) + i] < v) break;
      ++i;
      const int up = min(__ffs(i) - 1, log - k);
      i >>= up;
      k += up;
    }
    while (k > 0) {
      --k;
      i <<= 1;
      if (m[off(k) + i] >= v) ++i;
    }
    return i;
  }
  // nearest tile t' <= s with m[t'] < v, -1 if there is none
  __device__ __forceinline__ int left(int s, uint32_t v) const {
    int i = s, k = 0;
    while (true) {
      if (i < 0) return -1;
      if (m[off(k) + i] < v) break;
      --i;
      if (i < 0) return -1;
      const int up = min(__ffs(i + 1) - 1, log - k);
      i >>= up;
      k += up;
    }
    while (k > 0) {
      --k;
      i = 2 * i + 1;
      if (m[off(k) + i] >= v) --i;
    }
    return i;
  }
};

// One of the 38 independent pieces of the box of the sorted leaves [l, r), l < r: pieces 0..13 are the
// ragged ends (< 8 leaves each, or all of a range without an aligned block of 8) read from the spheres,
// piece 14 + j is level PYR_BASE + j of the global pyramid (at most two entries per level).  The
// addresses depend only on l and r, so a warp issues all pieces of a node's two child boxes at once.
constexpr int RANGE_PIECES = 14 + (PYR_MAX_LEVELS - PYR_BASE + 1);
__device__ __forceinline__ void range_piece(const float4* __restrict__ sphere, const uint4* __restrict__ pyr, const QFrame& qf,
                                            uint32_t l, uint32_t r, int piece, QBox& A) {
  const uint32_t lb = (l + (1u << PYR_BASE) - 1) >> PYR_BASE, rb = r >> PYR_BASE;
  const bool small = lb >= rb;   // no aligned block inside: < 2 x 8 leaves, all read directly
  if (piece < 14) {
    uint32_t i;
    if (small) i = l + piece;
    else if (piece < 7) { i = l + piece; if (i >= (lb << PYR_BASE)) return; }
    else i = (rb << PYR_BASE) + (piece - 7);
    if (i < r) A.merge(quant_sphere(__ldg(sphere + i), qf));
    return;
  }
  if (small) return;
  const int k = PYR_BASE + (piece - 14);
  const uint32_t lk = (l + (1u << k) - 1) >> k, rk = r >> k;   // the segment-tree walk's bounds when it reaches level k
  if (lk >= rk) return;
  const uint4* lev = pyr + (size_t)c_pyr.off[k];
  if (lk & 1u) {
    const uint4 e = __ldg(lev + lk);
    QBox b; b.w[0] = e.x; b.w[1] = e.y; b.w[2] = e.z;
    A.merge(b);
  }
  if (rk & 1u) {
    const uint4 e = __ldg(lev + (rk - 1));
    QBox b; b.w[0] = e.x; b.w[1] = e.y; b.w[2] = e.z;
    A.merge(b);
  }
}

// One warp per queued node; persistent blocks (the per-tile minima are staged once per block).
constexpr int SPINE_THREADS = 256;
#ifndef SPLATS_SPINE_LANES
#define SPLATS_SPINE_LANES 8
#endif
constexpr int SPINE_LANES = SPLATS_SPINE_LANES;   // 32, 16 or 8
__global__ void __launch_bounds__(SPINE_THREADS)
tree_spine_kernel(const uint64_t* __restrict__ keys, FrameState* st, const int4* __restrict__ queue,
                  const float4* __restrict__ sphere, const uint4* __restrict__ pyr, QNode* __restrict__ qnodes,
                  const uint8_t* __restrict__ tile_min, const uint16_t* __restrict__ tile_fb, int nt_log) {
  pdl_wait();
#if SPLATS_LATE_TRIGGER < 3
  pdl_trigger();
#endif
  extern __shared__ __align__(16) unsigned char spine_smem[];
  uint8_t* m = spine_smem;
  const int n = (int)st->n;
  const int qn = (int)st->spine_n;
  constexpr int WPB = SPINE_THREADS / 32;
  if ((int)(blockIdx.x * WPB * (32 / SPINE_LANES)) >= qn) return;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int ntiles = (n + TT_LEAVES - 1) / TT_LEAVES;
  const QFrame qf = load_qframe(st);
  TileMins tm;
  tm.m = m;
  tm.log = nt_log;
  tm.nt = 1 << nt_log;
  for (int t = threadIdx.x; t < tm.nt; t += SPINE_THREADS) m[t] = t < ntiles ? __ldg(tile_min + t) : (uint8_t)255;
  __syncthreads();
  for (int k = 1; k <= tm.log; ++k) {
    const int cnt = tm.nt >> k, o0 = tm.off(k - 1), o1 = tm.off(k);
    for (int j = threadIdx.x; j < cnt; j += SPINE_THREADS) m[o1 + j] = min(m[o0 + 2 * j], m[o0 + 2 * j + 1]);
    __syncthreads();
  }
  // SPINE_LANES lanes per queued node (a warp works on 32 / SPINE_LANES nodes at once: the kernel is a chain of
  // three dependent round trips per node, so nodes in flight are what counts)
  constexpr int GPW = 32 / SPINE_LANES;                 // groups per warp
  const int sub = lane / SPINE_LANES, sl = lane % SPINE_LANES;
  const int stride = gridDim.x * WPB * GPW;
  for (int e0 = (blockIdx.x * WPB + warp) * GPW; e0 < qn; e0 += stride) {
    const int e = e0 + sub;
    const bool act = e < qn;
    // ---- the node's range (every lane of the group computes the same values: broadcast loads)
    const int4 ent = act ? __ldg(queue + e) : make_int4(0, 0, 0, 1);
    const int g = ent.x, t = g >> TT_LOG;
    const uint32_t v = (uint32_t)ent.w;
    int first = ent.y, last = ent.z;
    if (act && first < 0) {   // nearest split to the left, in an earlier tile, with a smaller delta
      const int t2 = tm.left(t - 1, v);
      first = t2 < 0 ? 0 : (t2 << TT_LOG) + (int)__ldg(tile_fb + (size_t)t2 * (2 * TT_VPAD) + TT_VPAD + v) + 1;
    }
    if (act && last < 0) {    // the array ends with a split of delta + 1 = 0, so there always is one
      const int t2 = tm.right(t + 1, v);
      last = (t2 << TT_LOG) + (int)__ldg(tile_fb + (size_t)t2 * (2 * TT_VPAD) + v);
    }
    // ---- both child boxes: 2 x RANGE_PIECES independent pieces spread over the group's lanes, then a reduction
    QBox L, R;
    L.init();
    R.init();
    if (act) {
      for (int piece = sl; piece < 2 * RANGE_PIECES; piece += SPINE_LANES) {
        if (piece < RANGE_PIECES) range_piece(sphere, pyr, qf, (uint32_t)first, (uint32_t)g + 1u, piece, L);
        else range_piece(sphere, pyr, qf, (uint32_t)g + 1u, (uint32_t)last + 1u, piece - RANGE_PIECES, R);
      }
    }
    int idx = 0;
    if (act) {
      const int dl = first > 0 ? delta(keys, n, first - 1, __ldg(keys + first - 1), first) : -1;
      const int dr = last < n - 1 ? delta(keys, n, last, __ldg(keys + last), last + 1) : -1;
      idx = dr > dl ? last : first;
    }
#pragma unroll
    for (int o = SPINE_LANES / 2; o > 0; o >>= 1) {
      L.merge(L.shfl_xor(o));
      R.merge(R.shfl_xor(o));
    }
    if (act && sl == 0) {
      const int cnt_l = g - first + 1, cnt_r = last - g;
      const int left = cnt_l <= LEAF_MAX ? (int)leaf_range_code((uint32_t)first, (uint32_t)cnt_l) : g;
      const int right = cnt_r <= LEAF_MAX ? (int)leaf_range_code((uint32_t)g + 1u, (uint32_t)cnt_r) : g + 1;
      store_qnode(qnodes + idx, L, R, left, right);
    }
  }
}

}  // namespace sw
