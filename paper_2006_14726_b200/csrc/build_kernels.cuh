// build_kernels.cuh -- steps a1 (scene bounds) and a2 (unproject + validate + Morton +
// order-preserving compaction + digit histograms) of SURVEY.md sec. 8(a).
//
// Both kernels walk the source frame in the same tiles of TILE_PX consecutive pixels; a
// thread owns 8 consecutive pixels (two 16-byte vector loads of depth), so the compacted
// output keeps ascending pixel order, which makes the later stable sort an order by
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

// Where the splat centres come from.  FrameSource: the 2.5D frame itself (splats_update; Eq. 1
// per valid pixel).  PackedSource: a received buffer of quantised samples (splats_update_packed;
// every element is a splat unless its radius field is 0).  Element index = splat id.
struct FrameSource {
  const float* __restrict__ depth;
  DevCamera cam;
  using Raw = float;
  __device__ __forceinline__ int width() const { return cam.W; }
  __device__ __forceinline__ void load8(int64_t base, int64_t P, Raw t[8]) const { load_depth8(depth, base, P, t); }
  __device__ __forceinline__ bool valid(Raw t) const { return depth_valid(t); }
  __device__ __forceinline__ void centre(Raw t, int x, int y, float p[3]) const {
    float len;
    splat_centre(cam, x, y, t, p, len);
  }
};
struct PackedSource {
  const uint64_t* __restrict__ samples;
  QuantParams q;
  using Raw = uint64_t;
  __device__ __forceinline__ int width() const { return 0x7fffffff; }  // one long row: x = index
  __device__ __forceinline__ void load8(int64_t base, int64_t P, Raw w[8]) const {
    if (base + 8 <= P) {
      const ulonglong2* v = reinterpret_cast<const ulonglong2*>(samples + base);
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        const ulonglong2 a = __ldg(v + k);
        w[2 * k] = a.x;
        w[2 * k + 1] = a.y;
      }
    } else {
#pragma unroll
      for (int k = 0; k < 8; ++k) w[k] = (base + k < P) ? __ldg(samples + base + k) : 0ull;
    }
  }
  __device__ __forceinline__ bool valid(Raw w) const { return (w >> 48) != 0ull; }
  __device__ __forceinline__ void centre(Raw w, int, int, float p[3]) const { decode_centre(w, q, p); }
};

// ------------------------------------------------------------------------------------ a1
// Scene bounds = component-wise min/max of the valid splat centres (Eq. 1),
// number of valid pixels per tile (for the compaction) and in total.
template <class Src>
__global__ void __launch_bounds__(BUILD_THREADS)
bounds_kernel(const Src src, int64_t P, FrameState* __restrict__ st, uint32_t* __restrict__ tile_count) {
  pdl_wait();
  pdl_trigger();
  __shared__ float s_red[6][BUILD_THREADS / 32];
  __shared__ uint32_t s_cnt[BUILD_THREADS / 32];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int64_t base = (int64_t)blockIdx.x * TILE_PX + (int64_t)tid * PX_PER_THREAD;
  const float INF = __int_as_float(0x7f800000);
  float lo[3] = {INF, INF, INF}, hi[3] = {-INF, -INF, -INF};
  uint32_t cnt = 0;
  if (base < P) {
    typename Src::Raw t[8];
    src.load8(base, P, t);
    const int W = src.width();
    int y = (int)(base / W), x = (int)(base - (int64_t)y * W);
#pragma unroll
    for (int k = 0; k < 8; ++k) {
      if (src.valid(t[k])) {
        float p[3];
        src.centre(t[k], x, y, p);
#pragma unroll
        for (int a = 0; a < 3; ++a) { lo[a] = fminf(lo[a], p[a]); hi[a] = fmaxf(hi[a], p[a]); }
        ++cnt;
      }
      if (++x == W) { x = 0; ++y; }
    }
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      lo[a] = fminf(lo[a], __shfl_xor_sync(0xffffffffu, lo[a], o));
      hi[a] = fmaxf(hi[a], __shfl_xor_sync(0xffffffffu, hi[a], o));
    }
    cnt += __shfl_xor_sync(0xffffffffu, cnt, o);
  }
  if (lane == 0) {
#pragma unroll
    for (int a = 0; a < 3; ++a) { s_red[a][warp] = lo[a]; s_red[3 + a][warp] = hi[a]; }
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
#pragma unroll
    for (int o = NW / 2; o > 0; o >>= 1) {
#pragma unroll
      for (int a = 0; a < 3; ++a) {
        lo[a] = fminf(lo[a], __shfl_xor_sync(0xffffffffu, lo[a], o));
        hi[a] = fmaxf(hi[a], __shfl_xor_sync(0xffffffffu, hi[a], o));
      }
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
        atomicAdd(&st->n, cnt);
      }
    }
  }
}

// ------------------------------------------------------------------------------------ a2
__device__ __forceinline__ uint64_t spread21(uint32_t v) {  // bit i -> bit 3i
  uint64_t x = v & 0x1fffffu;
  x = (x | (x << 32)) & 0x001f00000000ffffull;
  x = (x | (x << 16)) & 0x001f0000ff0000ffull;
  x = (x | (x << 8)) & 0x100f00f00f00f00full;
  x = (x | (x << 4)) & 0x10c30c30c30c30c3ull;
  x = (x | (x << 2)) & 0x1249249249249249ull;
  return x;
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

// Persistent over tiles.  Per tile: offset = sum of the valid counts of all earlier tiles,
// block scan of the per-thread counts, keys/ids written in pixel order.  The eight 8-bit
// digit histograms of the radix sort are accumulated in shared memory on the way (the keys
// are in registers anyway) and flushed once per block.  Block 0 also re-arms the other
// parity's FrameState for the next frame.
template <class Src>
__global__ void __launch_bounds__(BUILD_THREADS)
unproject_kernel(const Src src, int64_t P, int num_tiles,
                 FrameState* __restrict__ st, FrameState* __restrict__ st_next,
                 const uint32_t* __restrict__ tile_count, uint64_t* __restrict__ keys0,
                 uint32_t* __restrict__ ids0, uint64_t* __restrict__ keys1, uint32_t* __restrict__ ids1,
                 int sort_mode) {
  pdl_wait();
  pdl_trigger();
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
#pragma unroll
    for (int d = 0; d < 8; ++d) st_next->hist[d][tid] = 0u;
  }
#pragma unroll
  for (int d = 0; d < 8; ++d) s_hist[d][tid] = 0u;

  // the sort ping-pongs between two buffers and must end in buffer 0 (onesweep.cuh)
  const bool odd = sort_input_buffer(sort_mode, st->n) != 0;
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

    const int64_t base = (int64_t)tile * TILE_PX + (int64_t)tid * PX_PER_THREAD;
    uint64_t code[8];
    uint32_t vmask = 0;
    if (base < P && tile_count[tile] != 0) {
      typename Src::Raw t[8];
      src.load8(base, P, t);
      const int W = src.width();
      int y = (int)(base / W), x = (int)(base - (int64_t)y * W);
#pragma unroll
      for (int k = 0; k < 8; ++k) {
        if (src.valid(t[k])) {
          float p[3];
          src.centre(t[k], x, y, p);
          code[k] = morton63(p, lo, ext);
          vmask |= 1u << k;
        }
        if (++x == W) { x = 0; ++y; }
      }
    }
    // block exclusive scan of popc(vmask)
    uint32_t c = __popc(vmask), incl = c;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      uint32_t n = __shfl_up_sync(0xffffffffu, incl, o);
      if (lane >= o) incl += n;
    }
    if (lane == 31) s_warp[warp] = incl;
    __syncthreads();
    uint32_t tile_off = 0, warp_off = 0;
#pragma unroll
    for (int w = 0; w < NW; ++w) {
      tile_off += s_part[w];
      if (w < warp) warp_off += s_warp[w];
    }
    uint32_t pos = tile_off + warp_off + incl - c;
#pragma unroll
    for (int k = 0; k < 8; ++k) {
      const bool v = (vmask >> k) & 1u;
      if (v) {
        keys[pos] = code[k];
        ids[pos] = (uint32_t)(base + k);
        ++pos;
      }
      // digit histograms; the high digits are warp-coherent (neighbouring pixels share the
      // coarse cell), so aggregate them with match_any before touching shared memory
      const unsigned act = __ballot_sync(0xffffffffu, v);
      if (v) {
#pragma unroll
        for (int d = 0; d < 4; ++d) atomicAdd(&s_hist[d][(code[k] >> (8 * d)) & 0xff], 1u);
#pragma unroll
        for (int d = 4; d < 8; ++d) {
          const uint32_t dig = (uint32_t)(code[k] >> (8 * d)) & 0xff;
          const unsigned peers = __match_any_sync(act, dig);
          if ((peers & ((1u << lane) - 1)) == 0) atomicAdd(&s_hist[d][dig], (uint32_t)__popc(peers));
        }
      }
    }
    __syncthreads();  // s_warp / s_part reused by the next tile
  }
  __syncthreads();
#pragma unroll
  for (int d = 0; d < 8; ++d) {
    const uint32_t h = s_hist[d][tid];
    if (h) atomicAdd(&st->hist[d][tid], h);
  }
}

}  // namespace sw
