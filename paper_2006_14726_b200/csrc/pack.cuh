// pack.cuh -- server side of the paper's wire format: the 2.5D frame
// becomes a compacted buffer of 64-bit object-space samples plus 32-bit colours.
//
// "We quantize the object space coordinate and pack it together with the radius into
// 64 bits. ... Before sending we compact that buffer by moving all the samples with zero radius
// to one side and send only those object space samples with non-zero radius."  The paper does
// this compaction serially on the CPU (23 ms for 1024 x 1024, Table 1) and names it
// the bottleneck of its pipeline (where it suggests thrust::remove_if); here it is
// two bandwidth-bound launches that keep ascending pixel order.
#pragma once
#include "build_kernels.cuh"

namespace sw {

struct PackArgs {
  const float4* __restrict__ color;
  const float* __restrict__ depth;
  DevCamera cam;
  RadiusParams rp;
  QuantParams q;
  int64_t P;
  int num_tiles;
};

// Eq. 1 + radius for pixel idx; false if the pixel is dropped (invalid depth or
// zero radius).  The colour is only fetched when it is needed.
__device__ __forceinline__ bool pack_pixel(const PackArgs& a, int64_t idx, int x, int y, float t, bool want_words,
                                           uint64_t& word, uint32_t& c8) {
  if (!depth_valid(t)) return false;
  float p[3], len;
  splat_centre(a.cam, x, y, t, p, len);
  const float z = div_(t, len);
  float4 col = make_float4(0.f, 0.f, 0.f, 0.f);
  if (want_words || a.rp.mode == 2) col = ldg_stream_f4(a.color + idx);
  const float r = splat_radius(a.rp, z, col.w);
  if (!(r > 0.0f)) return false;
  if (want_words) {
    word = pack_sample(p, r, a.q);
    c8 = pack_colour(col);
  }
  return true;
}

// Number of kept samples per tile of TILE_PX pixels.
__global__ void __launch_bounds__(BUILD_THREADS)
pack_count_kernel(const PackArgs a, uint32_t* __restrict__ tile_count) {
  __shared__ uint32_t s_cnt[BUILD_THREADS / 32];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int64_t base = (int64_t)blockIdx.x * TILE_PX + (int64_t)tid * PX_PER_THREAD;
  uint32_t cnt = 0;
  if (base < a.P) {
    float t[8];
    load_depth8(a.depth, base, a.P, t);
    int y = (int)(base / a.cam.W), x = (int)(base - (int64_t)y * a.cam.W);
#pragma unroll
    for (int k = 0; k < 8; ++k) {
      uint64_t w;
      uint32_t c;
      cnt += pack_pixel(a, base + k, x, y, t[k], false, w, c) ? 1u : 0u;
      if (++x == a.cam.W) { x = 0; ++y; }
    }
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) cnt += __shfl_xor_sync(0xffffffffu, cnt, o);
  if (lane == 0) s_cnt[warp] = cnt;
  __syncthreads();
  if (tid == 0) {
    uint32_t tot = 0;
#pragma unroll
    for (int w = 0; w < BUILD_THREADS / 32; ++w) tot += s_cnt[w];
    tile_count[blockIdx.x] = tot;
  }
}

// Persistent over tiles: offset = sum of the counts of all earlier tiles, block scan of the
// per-thread counts, samples and colours written in pixel order.  The block that owns the last
// tile also writes the total.
__global__ void __launch_bounds__(BUILD_THREADS)
pack_write_kernel(const PackArgs a, const uint32_t* __restrict__ tile_count, uint64_t* __restrict__ samples,
                  uint32_t* __restrict__ colours, uint32_t* __restrict__ count_out) {
  __shared__ uint32_t s_warp[BUILD_THREADS / 32];
  __shared__ uint32_t s_part[BUILD_THREADS / 32];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  constexpr int NW = BUILD_THREADS / 32;
  for (int tile = blockIdx.x; tile < a.num_tiles; tile += gridDim.x) {
    uint32_t part = 0;
    for (int i = tid; i < tile; i += BUILD_THREADS) part += tile_count[i];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) part += __shfl_xor_sync(0xffffffffu, part, o);
    if (lane == 0) s_part[warp] = part;

    const int64_t base = (int64_t)tile * TILE_PX + (int64_t)tid * PX_PER_THREAD;
    const uint32_t tile_total = tile_count[tile];
    uint64_t word[8];
    uint32_t c8[8];
    uint32_t vmask = 0;
    if (base < a.P && tile_total != 0) {
      float t[8];
      load_depth8(a.depth, base, a.P, t);
      int y = (int)(base / a.cam.W), x = (int)(base - (int64_t)y * a.cam.W);
#pragma unroll
      for (int k = 0; k < 8; ++k) {
        if (pack_pixel(a, base + k, x, y, t[k], true, word[k], c8[k])) vmask |= 1u << k;
        if (++x == a.cam.W) { x = 0; ++y; }
      }
    }
    const uint32_t c = __popc(vmask);
    uint32_t incl = c;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const uint32_t n = __shfl_up_sync(0xffffffffu, incl, o);
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
      if ((vmask >> k) & 1u) {
        samples[pos] = word[k];
        colours[pos] = c8[k];
        ++pos;
      }
    }
    if (tile == a.num_tiles - 1 && tid == 0) *count_out = tile_off + tile_total;
    __syncthreads();  // s_warp / s_part reused by the next tile
  }
}

}  // namespace sw
