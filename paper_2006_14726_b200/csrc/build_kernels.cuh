// build_kernels.cuh -- steps a1 (scene bounds) and a2 (unproject + validate + Morton +
// order-preserving compaction + digit histograms) of SURVEY.md sec. 8(a).
//
// Both kernels walk the source frame in the same tiles of TILE_PX consecutive pixels and keep
// ascending pixel order in the compacted output, which makes the later stable sort an order by
// (code, id) (north_star: "keyed on (code, splat id) so ties are stable and deterministic").
#pragma once
#include "common.cuh"

namespace sw {

constexpr int BUILD_THREADS = 256;
constexpr int PX_PER_THREAD = 8;
constexpr int TILE_PX = BUILD_THREADS * PX_PER_THREAD;  // 2048

// Load the 8 depths a thread owns (vector path when the whole group is in range).
__device__ __forceinline__ void load_depth8(const float* __restrict__ depth, int64_t base, int64_t P, float t[8]) {
  if (base + 8 <= P) {
    float4 a = ldg_stream_f4(reinterpret_cast<const float4*>(depth + base));
    float4 b = ldg_stream_f4(reinterpret_cast<const float4*>(depth + base + 4));
    t[0] = a.x; t[1] = a.y; t[2] = a.z; t[3] = a.w;
    t[4] = b.x; t[5] = b.y; t[6] = b.z; t[7] = b.w;
  } else {
#pragma unroll
    for (int k = 0; k < 8; ++k) t[k] = (base + k < P) ? __ldg(depth + base + k) : 0.0f;
  }
}

// Where the splat centres come from.  FrameSource: the 2.5D frame itself (splats_update): Eq. 1 is
// evaluated ONCE per valid pixel, in bounds_kernel, which stores the splat (centre + radius) at its
// pixel index; unproject_kernel and the tree's gather read that record instead of evaluating Eq. 1
// again (three IEEE divisions + a square root + three more divisions per pixel each time).
// PackedSource: a received buffer of quantised samples (splats_update_packed; every element is a
// splat unless its radius field is 0); decoding is cheap, nothing is stored.  Element index = splat id.
struct FrameSource {
  const float* __restrict__ depth;
  const float4* __restrict__ color;   // alpha is read only by the opacity radius (RadiusParams mode 2)
  float4* sphere_px;                  // [P] splat of every valid pixel, written by bounds_kernel
  DevCamera cam;
  RadiusParams rp;
  using Raw = float;
  __device__ __forceinline__ int width() const { return cam.W; }
  __device__ __forceinline__ Raw load(int64_t i) const { return __ldg(depth + i); }
  __device__ __forceinline__ Raw invalid() const { return 0.0f; }
  __device__ __forceinline__ bool valid(Raw t) const { return depth_valid(t); }
  __device__ __forceinline__ float bounds_centre(Raw t, int64_t i, int x, int y, float p[3]) const {   // returns the radius
    float len;
    splat_centre(cam, x, y, t, p, len);
    const float z = div_(t, len);
    const float alpha = rp.mode == 2 ? __ldg(&color[i].w) : 0.0f;
    const float r = splat_radius(rp, z, alpha);
    sphere_px[i] = make_float4(p[0], p[1], p[2], r);
    return r;
  }
  __device__ __forceinline__ void key_centre(Raw, int64_t i, float p[3]) const {
    const float4 sp = __ldcg(sphere_px + i);   // written by the previous kernel of this stream
    p[0] = sp.x; p[1] = sp.y; p[2] = sp.z;
  }
};
struct PackedSource {
  const uint64_t* __restrict__ samples;
  QuantParams q;
  using Raw = uint64_t;
  __device__ __forceinline__ int width() const { return 0x7fffffff; }  // one long row: x = index
  __device__ __forceinline__ Raw load(int64_t i) const { return __ldg(samples + i); }
  __device__ __forceinline__ Raw invalid() const { return 0ull; }
  __device__ __forceinline__ bool valid(Raw w) const { return (w >> 48) != 0ull; }
  __device__ __forceinline__ float bounds_centre(Raw w, int64_t, int, int, float p[3]) const {
    decode_centre(w, q, p);
    return decode_radius(w, q);
  }
  __device__ __forceinline__ void key_centre(Raw w, int64_t, float p[3]) const { decode_centre(w, q, p); }
};

// Both kernels walk the source in tiles of TILE_PX consecutive elements; a warp owns 256 consecutive
// ones and visits them in 8 rounds of 32 (lane = consecutive element: every load and store of a
// round is one coalesced request, and a ballot gives the order-preserving rank).
constexpr int WARP_PX = TILE_PX / (BUILD_THREADS / 32);   // 256
constexpr int ROUNDS = WARP_PX / 32;                      // 8

// ------------------------------------------------------------------------------------ a1
// Scene bounds = component-wise min/max of the valid splat centres (Eq. 1), the
// largest radius (with the bounds: the frame of the quantised node boxes, common.cuh QNode),
// number of valid pixels per tile (for the compaction) and in total.
template <class Src>
__global__ void __launch_bounds__(BUILD_THREADS, 6)
bounds_kernel(const Src src, int64_t P, FrameState* __restrict__ st, uint32_t* __restrict__ tile_count, int wait_at_start) {
  // wait_at_start = 0: the kernel before this one in the stream is a render.  Nothing here touches
  // what a render reads or writes (it reads the caller's frame and writes the next frame's state,
  // the tile counts and the per-pixel splats, all of which the previous update has finished with:
  // the render's blocks only start after that update is complete), so the blocks may run under the
  // render's tail; one thread waits at the end so that this kernel still completes after it.
  if (wait_at_start) pdl_wait();
  pdl_trigger();
  __shared__ float s_red[7][BUILD_THREADS / 32];
  __shared__ uint32_t s_cnt[BUILD_THREADS / 32];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int64_t base = (int64_t)blockIdx.x * TILE_PX + (int64_t)warp * WARP_PX + lane;
  const float INF = __int_as_float(0x7f800000);
  float lo[3] = {INF, INF, INF}, hi[3] = {-INF, -INF, -INF}, rmax = 0.0f;
  uint32_t cnt = 0;
  typename Src::Raw t[ROUNDS];
#pragma unroll
  for (int k = 0; k < ROUNDS; ++k) t[k] = base + 32 * k < P ? src.load(base + 32 * k) : src.invalid();
  const int W = src.width();
  int y = (int)(base / W), x = (int)(base - (int64_t)y * W);
#pragma unroll
  for (int k = 0; k < ROUNDS; ++k) {
    if (src.valid(t[k])) {
      float p[3];
      rmax = fmaxf(rmax, src.bounds_centre(t[k], base + 32 * k, x, y, p));
#pragma unroll
      for (int a = 0; a < 3; ++a) { lo[a] = fminf(lo[a], p[a]); hi[a] = fmaxf(hi[a], p[a]); }
      ++cnt;
    }
    x += 32;
    while (x >= W) { x -= W; ++y; }
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      lo[a] = fminf(lo[a], __shfl_xor_sync(0xffffffffu, lo[a], o));
      hi[a] = fmaxf(hi[a], __shfl_xor_sync(0xffffffffu, hi[a], o));
    }
    rmax = fmaxf(rmax, __shfl_xor_sync(0xffffffffu, rmax, o));
    cnt += __shfl_xor_sync(0xffffffffu, cnt, o);
  }
  if (lane == 0) {
#pragma unroll
    for (int a = 0; a < 3; ++a) { s_red[a][warp] = lo[a]; s_red[3 + a][warp] = hi[a]; }
    s_red[6][warp] = rmax;
    s_cnt[warp] = cnt;
  }
  __syncthreads();
  if (warp == 0) {
    constexpr int NW = BUILD_THREADS / 32;
    cnt = lane < NW ? s_cnt[lane] : 0;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      lo[a] = lane < NW ? s_red[a][lane] : INF;
      hi[a] = lane < NW ? s_red[3 + a][lane] : -INF;
    }
    rmax = lane < NW ? s_red[6][lane] : 0.0f;
#pragma unroll
    for (int o = NW / 2; o > 0; o >>= 1) {
#pragma unroll
      for (int a = 0; a < 3; ++a) {
        lo[a] = fminf(lo[a], __shfl_xor_sync(0xffffffffu, lo[a], o));
        hi[a] = fmaxf(hi[a], __shfl_xor_sync(0xffffffffu, hi[a], o));
      }
      rmax = fmaxf(rmax, __shfl_xor_sync(0xffffffffu, rmax, o));
      cnt += __shfl_xor_sync(0xffffffffu, cnt, o);
    }
    if (lane == 0) {
      tile_count[blockIdx.x] = cnt;
      if (cnt) {
#pragma unroll
        for (int a = 0; a < 3; ++a) {
          atomicMin(&st->lo[a], f2ord(lo[a]));
          atomicMax(&st->hi[a], f2ord(hi[a]));
        }
        atomicMax(&st->rmax, f2ord(rmax));
        atomicAdd(&st->n, cnt);
      }
    }
  }
  if (!wait_at_start && tid == 0) pdl_wait();
}

// ------------------------------------------------------------------------------------ a2
__device__ __forceinline__ uint32_t spread11(uint32_t x) {  // bit i -> bit 3i, 11 bits (32-bit operations)
  x = (x | (x << 16)) & 0x070000ffu;
  x = (x | (x << 8)) & 0x0700f00fu;
  x = (x | (x << 4)) & 0x430c30c3u;
  x = (x | (x << 2)) & 0x49249249u;
  return x;
}
__device__ __forceinline__ uint64_t spread21(uint32_t v) {  // bit i -> bit 3i: low 11 bits and high 10 bits on their own
  return (uint64_t)spread11(v & 0x7ffu) | ((uint64_t)spread11((v >> 11) & 0x3ffu) << 33);
}

// 63-bit Morton code of centre p inside [lo, hi] (LBVH, PAPER.md:71 [LGS*09]); 21 bit per
// axis, x in the highest slot; a zero-extent axis quantises to 0.
__device__ __forceinline__ uint64_t morton63(const float p[3], const float lo[3], const float ext[3]) {
  uint32_t q[3];
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    if (ext[a] > 0.0f) {
      float s = mul_(div_(sub_(p[a], lo[a]), ext[a]), 2097152.0f);
      uint32_t v = __float2uint_rz(s);
      q[a] = v < 2097151u ? v : 2097151u;
    } else {
      q[a] = 0;
    }
  }
  return (spread21(q[0]) << 2) | (spread21(q[1]) << 1) | spread21(q[2]);
}

// Persistent over tiles.  Per tile: offset = sum of the valid counts of all earlier tiles, ranks
// from ballots (pixel order is kept), keys/ids written in pixel order.  The digit histograms that
// the chosen sort mode consumes are accumulated in shared memory on the way and flushed once per
// block: the hybrid sort reads only digits first..7 (the top 31 / 39 code bits; if it has to fall
// back to all eight passes it counts the low digits itself, onesweep.cuh); a warp's 32 lanes hold
// 32 consecutive pixels whose high digits mostly agree, so runs of equal digits are counted once.
// Block 0 also re-arms the next frame's FrameState.
template <class Src>
__global__ void __launch_bounds__(BUILD_THREADS, 6)
unproject_kernel(const Src src, int64_t P, int num_tiles,
                 FrameState* __restrict__ st, FrameState* __restrict__ st_next,
                 const uint32_t* __restrict__ tile_count, uint64_t* __restrict__ keys0,
                 uint32_t* __restrict__ ids0, uint64_t* __restrict__ keys1, uint32_t* __restrict__ ids1,
                 int sort_mode) {
  pdl_wait();
#if SPLATS_LATE_TRIGGER < 2
  pdl_trigger();
#endif
  __shared__ uint32_t s_hist[8][256];
  __shared__ uint32_t s_warp[BUILD_THREADS / 32];
  __shared__ uint32_t s_part[BUILD_THREADS / 32];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  constexpr int NW = BUILD_THREADS / 32;

  if (blockIdx.x == 0) {  // re-arm the accumulators of the next frame (other parity)
    if (tid < 3) { st_next->lo[tid] = 0xffffffffu; st_next->hi[tid] = 0u; }
    if (tid == 3) st_next->n = 0u;
    if (tid == 4) st_next->pyr_done = 0u;
    if (tid == 5) st_next->sort_bar = 0u;
    if (tid == 6) st_next->sort_fallback = 0u;
    if (tid == 7) st_next->spine_n = 0u;
    if (tid == 8) st_next->rmax = 0u;
    if (tid == 9) st_next->tile_done = 0u;
    if (tid == 10) st_next->sort_wfall = 0u;
#pragma unroll
    for (int d = 0; d < 8; ++d) st_next->hist[d][tid] = 0u;
  }
  if (blockIdx.x == 0 && tid == 32) {   // bounds and largest radius are final: the frame of the quantised node boxes
    const QFrame q = derive_qframe(st);
    const float rmax = ord2f(st->rmax);
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      st->qf[a] = q.lo[a]; st->qf[3 + a] = q.s[a]; st->qf[6 + a] = q.c[a];
      // the frame is also the scene box the renders cull against (the tiled build carries quantised boxes only;
      // the pyramid / atomic refit modes overwrite it with the exact root box)
      st->root_lo[a] = q.lo[a];
      st->root_hi[a] = add_(ord2f(st->hi[a]), rmax);
    }
  }
#pragma unroll
  for (int d = 0; d < 8; ++d) s_hist[d][tid] = 0u;

  // the sort ping-pongs between two buffers and must end in buffer 0 (onesweep.cuh)
  const uint32_t n_all = st->n;
  const bool odd = sort_input_buffer(sort_mode, n_all) != 0;
  // lowest digit whose histogram the sort launch reads from here (it counts any others itself, on its fallback paths)
  const int first_digit = sort_mode == SORT_HYBRID ? 8 - win_passes(n_all) : sort_mode == SORT_HYBRID_LSD ? hybrid_first_digit(n_all) : 0;
  uint64_t* __restrict__ keys = odd ? keys1 : keys0;
  uint32_t* __restrict__ ids = odd ? ids1 : ids0;
  float lo[3], ext[3];
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    lo[a] = ord2f(st->lo[a]);
    ext[a] = sub_(ord2f(st->hi[a]), lo[a]);
  }
  __syncthreads();

  for (int tile = blockIdx.x; tile < num_tiles; tile += gridDim.x) {
    // exclusive prefix of the tile counts (block reduce of tile_count[0..tile))
    uint32_t part = 0;
    for (int i = tid; i < tile; i += BUILD_THREADS) part += tile_count[i];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) part += __shfl_xor_sync(0xffffffffu, part, o);
    if (lane == 0) s_part[warp] = part;

    const int64_t base = (int64_t)tile * TILE_PX + (int64_t)warp * WARP_PX + lane;
    typename Src::Raw t[ROUNDS];
    uint32_t vmask = 0, wtotal = 0;
    const bool any = tile_count[tile] != 0;
    if (any) {
#pragma unroll
      for (int k = 0; k < ROUNDS; ++k) t[k] = base + 32 * k < P ? src.load(base + 32 * k) : src.invalid();
#pragma unroll
      for (int k = 0; k < ROUNDS; ++k) {
        const bool v = src.valid(t[k]);
        vmask |= (v ? 1u : 0u) << k;
        wtotal += __popc(__ballot_sync(0xffffffffu, v));
      }
    }
    if (lane == 0) s_warp[warp] = wtotal;
    __syncthreads();
    uint32_t pos = 0;
#pragma unroll
    for (int w = 0; w < NW; ++w) {
      pos += s_part[w];
      if (w < warp) pos += s_warp[w];
    }
    if (any) {
#pragma unroll
      for (int k = 0; k < ROUNDS; ++k) {
        const bool v = (vmask >> k) & 1u;
        const unsigned act = __ballot_sync(0xffffffffu, v);
        uint64_t code = 0;
        if (v) {
          float p[3];
          src.key_centre(t[k], base + 32 * k, p);
          // the sort key is the 63-bit code shifted up by one: all 64 bits carry information, the top digit has eight
          // significant bits instead of seven (one more bit per pass of the hybrid sorts; splats_export shifts back)
          code = morton63(p, lo, ext) << 1;
          const uint32_t at = pos + __popc(act & ((1u << lane) - 1));
          keys[at] = code;
          ids[at] = (uint32_t)(base + 32 * k);
        }
        // digit histograms: neighbouring pixels mostly share their top digits, so each run of equal digits among
        // consecutive valid lanes is counted by its first lane (one shared-memory atomic per run and digit)
        if (first_digit == 5) {
          // the windowed sort reads the digits 5 .. 7 only (up to 2^23 splats): runs of equal top 24 key bits, found once for all three
          const uint32_t top = v ? (uint32_t)(code >> 40) : 0xffffffffu;
          const uint32_t prev = __shfl_up_sync(0xffffffffu, top, 1);
          const bool head = v && (lane == 0 || prev != top);
          const unsigned brk = __ballot_sync(0xffffffffu, head || !v);   // where runs start or are interrupted
          if (head) {
            const unsigned after = lane == 31 ? 0u : brk >> (lane + 1);
            const uint32_t run = after ? (uint32_t)__ffs(after) : 32u - lane;
            atomicAdd(&s_hist[5][top & 0xff], run);
            atomicAdd(&s_hist[6][(top >> 8) & 0xff], run);
            atomicAdd(&s_hist[7][top >> 16], run);
          }
        } else {
          for (int d = first_digit; d < 8; ++d) {
            const uint32_t dig = v ? (uint32_t)(code >> (8 * d)) & 0xff : 0x100u;
            const uint32_t prev = __shfl_up_sync(0xffffffffu, dig, 1);
            const bool head = v && (lane == 0 || prev != dig);
            const unsigned brk = __ballot_sync(0xffffffffu, head || !v);   // where runs start or are interrupted
            if (head) {
              const unsigned after = lane == 31 ? 0u : brk >> (lane + 1);
              const uint32_t run = after ? (uint32_t)__ffs(after) : 32u - lane;
              atomicAdd(&s_hist[d][dig], run);
            }
          }
        }
        pos += __popc(act);
      }
    }
    __syncthreads();  // s_warp / s_part reused by the next tile
  }
  __syncthreads();
  for (int d = first_digit; d < 8; ++d) {
    const uint32_t h = s_hist[d][tid];
    if (h) atomicAdd(&st->hist[d][tid], h);
  }
}

}  // namespace sw
