// onesweep.cuh -- step a3: hand-written single-pass-per-digit LSD radix sort ("onesweep")
// of (63-bit Morton code, splat id) pairs, 8 bits per pass, stable (
// LBVH).
//
// One launch per digit.  The grid is persistent and co-resident (<= SMs x occupancy), tiles
// are dealt round-robin (block b owns tiles b, b+G, ...), and each tile obtains the global
// offset of each of its 256 digit bins by a chained scan with decoupled look-back over the
// tiles before it.  Because all blocks are resident and every block walks its tiles in
// ascending order, the lowest unfinished tile can always make progress: no deadlock, no
// atomic ticket.  The look-back status words carry an epoch (unique per pass and frame) so
// the status array never needs clearing.
//
// The digit histograms (hence the bin bases) come from unproject_kernel, which had the keys
// in registers anyway.
#pragma once
#include "common.cuh"

namespace sw {

constexpr int SORT_THREADS = 256;
constexpr int SORT_WARPS = SORT_THREADS / 32;
constexpr int RADIX = 256;

// status word: [63:32] epoch, [31:30] flag, [29:0] count
constexpr uint64_t FLAG_AGG = 1ull << 30;  // tile aggregate available
constexpr uint64_t FLAG_INC = 2ull << 30;  // inclusive prefix available
constexpr uint32_t VALUE_MASK = (1u << 30) - 1;

template <int ITEMS>
struct SortSmem {
  uint32_t warp_hist[SORT_WARPS][RADIX];  // per-warp digit counts -> exclusive prefix over warps
  uint32_t tile_off[RADIX];               // exclusive scan of the tile's digit counts
  int64_t bin_base[RADIX];                // global position of local slot 0 of each digit
  uint32_t digit_base[RADIX];             // exclusive scan of the global histogram
  uint32_t scan_tmp[SORT_WARPS];
  uint64_t stage[SORT_THREADS * ITEMS];   // keys (then values) in tile-sorted order
};

// exclusive scan of one value per thread over the 256-thread block
__device__ __forceinline__ uint32_t block_excl_scan_256(uint32_t v, uint32_t* tmp /*[8]*/, uint32_t* total) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  uint32_t incl = v;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    uint32_t n = __shfl_up_sync(0xffffffffu, incl, o);
    if (lane >= o) incl += n;
  }
  __syncthreads();  // tmp may still be read from a previous use
  if (lane == 31) tmp[warp] = incl;
  __syncthreads();
  uint32_t off = 0, tot = 0;
#pragma unroll
  for (int w = 0; w < SORT_WARPS; ++w) {
    uint32_t t = tmp[w];
    if (w < warp) off += t;
    tot += t;
  }
  if (total) *total = tot;
  return off + incl - v;
}

template <int ITEMS>
__global__ void __launch_bounds__(SORT_THREADS)
onesweep_kernel(const uint64_t* __restrict__ kin, const uint32_t* __restrict__ vin,
                uint64_t* __restrict__ kout, uint32_t* __restrict__ vout,
                const FrameState* __restrict__ st, int pass, uint64_t* __restrict__ status, uint32_t epoch) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  SortSmem<ITEMS>& s = *reinterpret_cast<SortSmem<ITEMS>*>(smem_raw);
  constexpr int TILE = SORT_THREADS * ITEMS;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const uint32_t n = st->n;
  const int num_tiles = (int)((n + TILE - 1) / TILE);
  if ((int)blockIdx.x >= num_tiles) return;
  const int shift = 8 * pass;
  const uint64_t ep = (uint64_t)epoch << 32;

  {  // bin bases of this digit: exclusive scan of the global histogram
    uint32_t h = st->hist[pass][tid];
    uint32_t e = block_excl_scan_256(h, s.scan_tmp, nullptr);
    s.digit_base[tid] = e;
  }

  for (int tile = blockIdx.x; tile < num_tiles; tile += gridDim.x) {
    const uint32_t tile_base = (uint32_t)tile * TILE;
    // ---- load, warp-striped: item (warp, j, lane) has index tile_base + warp*32*ITEMS + j*32 + lane
    uint64_t key[ITEMS];
    const uint32_t wbase = tile_base + warp * 32 * ITEMS + lane;
#pragma unroll
    for (int j = 0; j < ITEMS; ++j) {
      const uint32_t idx = wbase + j * 32;
      key[j] = idx < n ? kin[idx] : ~0ull;
    }
#pragma unroll
    for (int w = 0; w < SORT_WARPS; ++w) s.warp_hist[w][tid] = 0;
    __syncthreads();

    // ---- rank inside the warp, digit by digit, in index order (stable)
    uint32_t rank[ITEMS];
#pragma unroll
    for (int j = 0; j < ITEMS; ++j) {
      const bool valid = (wbase + j * 32) < n;
      const uint32_t dig = (uint32_t)(key[j] >> shift) & 0xff;
      const unsigned peers = __match_any_sync(0xffffffffu, valid ? dig : 0x100u);
      const uint32_t before = __popc(peers & ((1u << lane) - 1));
      uint32_t base = 0;
      if (valid) base = s.warp_hist[warp][dig];
      __syncwarp();
      if (valid && before == 0) s.warp_hist[warp][dig] = base + __popc(peers);
      __syncwarp();
      rank[j] = base + before;
    }
    __syncthreads();

    // ---- bin `tid`: exclusive prefix over the warps, tile count
    uint32_t count = 0;
#pragma unroll
    for (int w = 0; w < SORT_WARPS; ++w) {
      uint32_t c = s.warp_hist[w][tid];
      s.warp_hist[w][tid] = count;
      count += c;
    }
    const uint32_t toff = block_excl_scan_256(count, s.scan_tmp, nullptr);
    s.tile_off[tid] = toff;

    // ---- decoupled look-back for bin `tid`
    uint64_t* my = status + (size_t)tile * RADIX + tid;
    uint32_t excl;
    if (tile == 0) {
      excl = s.digit_base[tid];
    } else {
      st_volatile_u64(my, ep | FLAG_AGG | count);
      excl = 0;
      int t = tile - 1;
      while (true) {
        uint64_t w = ld_volatile_u64(status + (size_t)t * RADIX + tid);
        if ((w >> 32) != epoch || (w & (FLAG_AGG | FLAG_INC)) == 0) continue;  // not published yet
        excl += (uint32_t)w & VALUE_MASK;
        if (w & FLAG_INC) break;
        --t;
      }
    }
    st_volatile_u64(my, ep | FLAG_INC | (excl + count));
    s.bin_base[tid] = (int64_t)excl - (int64_t)toff;
    __syncthreads();

    // ---- scatter keys into tile-sorted order in shared memory, then out (coalesced runs)
    uint32_t slot[ITEMS];
#pragma unroll
    for (int j = 0; j < ITEMS; ++j) {
      const uint32_t dig = (uint32_t)(key[j] >> shift) & 0xff;
      const bool valid = (wbase + j * 32) < n;
      slot[j] = s.tile_off[dig] + s.warp_hist[warp][dig] + rank[j];
      if (valid) s.stage[slot[j]] = key[j];
    }
    __syncthreads();
    const uint32_t tile_n = min((uint32_t)TILE, n - tile_base);
    uint8_t odig[ITEMS];
#pragma unroll
    for (int j = 0; j < ITEMS; ++j) {
      const uint32_t k = tid + j * SORT_THREADS;
      if (k < tile_n) {
        const uint64_t kk = s.stage[k];
        odig[j] = (uint8_t)((kk >> shift) & 0xff);
        kout[s.bin_base[odig[j]] + k] = kk;
      }
    }
    __syncthreads();
    // ---- values the same way
    uint32_t* vstage = reinterpret_cast<uint32_t*>(s.stage);
#pragma unroll
    for (int j = 0; j < ITEMS; ++j) {
      const uint32_t idx = wbase + j * 32;
      if (idx < n) vstage[slot[j]] = vin[idx];
    }
    __syncthreads();
#pragma unroll
    for (int j = 0; j < ITEMS; ++j) {
      const uint32_t k = tid + j * SORT_THREADS;
      if (k < tile_n) vout[s.bin_base[odig[j]] + k] = vstage[k];
    }
    __syncthreads();
  }
}

}  // namespace sw
