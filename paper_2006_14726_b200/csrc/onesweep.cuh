// onesweep.cuh -- step a3: hand-written single-pass-per-digit LSD radix sort ("onesweep")
// of (63-bit Morton code, splat id) pairs, 8 bits per pass, stable (
// LBVH).
//
// The grid is persistent and co-resident (<= SMs x occupancy), tiles are dealt round-robin
// (block b owns tiles b, b+G, ...), and each tile obtains the global offset of each of its 256
// digit bins by a chained scan with decoupled look-back over the tiles before it.  Because all
// blocks are resident and every block walks its tiles in ascending order, the lowest
// unfinished tile can always make progress: no deadlock, no atomic ticket.  The look-back
// status words carry an epoch (unique per pass and frame) so the status array never needs
// clearing.  When every tile has its own resident block (one wave) the chain is replaced by a
// two-level sum (tile aggregates + group totals), see onesweep_pass.  The digit histograms (hence
// the bin bases) come from unproject_kernel, which had the keys in registers anyway.
//
// One launch runs several passes, separated by a grid barrier (the grid is co-resident
// anyway), in one of three modes:
//   SORT_HYBRID (default)  passes 4..7 only, i.e. a stable sort by the top 31 code bits (32..62); then
//       every block checks its tiles for neighbours with equal top bits.  For the frames
//       this library is made for (one sample per pixel of a surface: the 2048 x 1024 x 1024
//       cells of those bits are finer than the sample pitch) there are none and the
//       order is already the order by (code, id).  Short runs of equal top bits (<= RUN_MAX)
//       are put in order by a stable insertion sort on the full code; a longer run raises a
//       flag and the same launch then redoes the sort with all 8 passes (degenerate inputs:
//       many equal codes).  The result is the same permutation in every case.
//   SORT_LSD8     all 8 passes in one launch.
//   SORT_SINGLE   one pass per launch (8 launches), the classic arrangement.
// Within a launch a buffer is read in one pass and written in the next, so keys and values
// are read with ld.global.cg (L2): a line cached in L1 by an earlier pass would be stale.
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
#ifndef SPLATS_LOOKBACK
#define SPLATS_LOOKBACK 8
#endif
constexpr int LOOKBACK = SPLATS_LOOKBACK;
constexpr int RUN_MAX = 32;           // longest run of equal top bits fixed up in place

struct SortArgs {
  uint64_t* key[2];
  uint32_t* val[2];
  FrameState* st;
  uint64_t* status;
  uint32_t epoch0;   // this launch may use epochs epoch0 .. epoch0 + 11
  int mode;
  int pass;          // SORT_SINGLE: the digit; input buffer = pass & 1
};

#ifndef SPLATS_RANK_BALLOT
#define SPLATS_RANK_BALLOT 1
#endif
#ifndef SPLATS_SORT_MAX_ITEMS
#define SPLATS_SORT_MAX_ITEMS 16
#endif
constexpr int SORT_MAX_ITEMS = SPLATS_SORT_MAX_ITEMS;
struct SortSmem {
  uint32_t warp_hist[SORT_WARPS][RADIX];  // per-warp digit counts -> exclusive prefix over warps
  uint32_t tile_off[RADIX];               // exclusive scan of the tile's digit counts
  int64_t bin_base[RADIX];                // global position of local slot 0 of each digit
  uint32_t digit_base[RADIX];             // exclusive scan of the global histogram
  uint32_t scan_tmp[SORT_WARPS];
  uint64_t stage[SORT_THREADS * SORT_MAX_ITEMS];   // keys in tile-sorted order
  uint32_t vstage[SORT_THREADS * SORT_MAX_ITEMS];  // values in tile-sorted order
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

// Grid barrier over the nb participating blocks (all co-resident); `bar` only ever grows
// within a frame and is re-armed by unproject_kernel of the next frame.
__device__ __forceinline__ void grid_barrier(uint32_t* bar, uint32_t nb, uint32_t& round) {
  ++round;
  __syncthreads();
  if (threadIdx.x == 0) {
    __threadfence();
    atomicAdd(bar, 1u);
    while (*reinterpret_cast<volatile uint32_t*>(bar) < round * nb) {}
    __threadfence();
  }
  __syncthreads();
}

// One 8-bit pass over all tiles of this block: in -> out.
template <int ITEMS>
__device__ __forceinline__ void onesweep_pass(SortSmem& s, const uint64_t* kin, const uint32_t* vin,
                                              uint64_t* kout, uint32_t* vout, const FrameState* st, int pass,
                                              uint64_t* status, uint32_t epoch, uint32_t n, int num_tiles) {
  constexpr int TILE = SORT_THREADS * ITEMS;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int shift = 8 * pass;
  const uint64_t ep = (uint64_t)epoch << 32;
  const bool single_wave = num_tiles <= (int)gridDim.x;   // every tile has its own resident block
  int gs_log = 3;
  while ((1 << (2 * gs_log)) < num_tiles) ++gs_log;
  uint64_t* gstatus = status + (size_t)num_tiles * RADIX;   // group totals live behind the tiles' words

  {  // bin bases of this digit: exclusive scan of the global histogram
    uint32_t h = __ldcg(&st->hist[pass][tid]);
    uint32_t e = block_excl_scan_256(h, s.scan_tmp, nullptr);
    s.digit_base[tid] = e;
  }

  for (int tile = blockIdx.x; tile < num_tiles; tile += gridDim.x) {
    const uint32_t tile_base = (uint32_t)tile * TILE;
    // ---- load, warp-striped: item (warp, j, lane) has index tile_base + warp*32*ITEMS + j*32 + lane
    uint64_t key[ITEMS];
    uint32_t val[ITEMS];
    const uint32_t wbase = tile_base + warp * 32 * ITEMS + lane;
#pragma unroll
    for (int j = 0; j < ITEMS; ++j) {
      const uint32_t idx = wbase + j * 32;
      key[j] = idx < n ? __ldcg(kin + idx) : ~0ull;
    }
#pragma unroll
    for (int j = 0; j < ITEMS; ++j) {
      const uint32_t idx = wbase + j * 32;
      val[j] = idx < n ? __ldcg(vin + idx) : 0u;
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
#if SPLATS_RANK_BALLOT
      // lanes with the same digit, from eight ballots: fixed latency and pipelined, where MATCH.ANY takes
      // time in proportion to the number of distinct digits in the warp (about 30 of 32 here)
      unsigned peers = __ballot_sync(0xffffffffu, valid);
#pragma unroll
      for (int b = 0; b < 8; ++b) {
        // bit test into a predicate, ballot, then one of two predicated ANDs (the compiler's own version builds
        // a select mask per bit: 7 instructions instead of a ballot and two predicated ANDs)
        asm("{\n\t.reg .pred p;\n\t.reg .b32 t;\n\t"
            "and.b32 t, %1, %2;\n\tsetp.ne.u32 p, t, 0;\n\t"
            "vote.sync.ballot.b32 t, p, 0xffffffff;\n\t"
            "@p and.b32 %0, %0, t;\n\t"
            "@!p lop3.b32 %0, %0, t, 0, 0x30;\n\t}"   // peers & ~t
            : "+r"(peers) : "r"(dig), "r"(1u << b));
      }
#else
      const unsigned peers = __match_any_sync(0xffffffffu, valid ? dig : 0x100u);
#endif
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
    // ---- publish the aggregate, then scan the tile's counts while the status word travels
    uint64_t* my = status + (size_t)tile * RADIX + tid;
    if (tile != 0 || single_wave) st_volatile_u64(my, ep | FLAG_AGG | count);
    const uint32_t toff = block_excl_scan_256(count, s.scan_tmp, nullptr);
    s.tile_off[tid] = toff;
    __syncthreads();

    // ---- keys and values into tile-sorted order in shared memory: this needs only the tile's
    // own counts, so it is done before the look-back and frees the registers for it
#pragma unroll
    for (int j = 0; j < ITEMS; ++j) {
      const uint32_t dig = (uint32_t)(key[j] >> shift) & 0xff;
      if ((wbase + j * 32) < n) {
        const uint32_t slot = s.tile_off[dig] + s.warp_hist[warp][dig] + rank[j];
        s.stage[slot] = key[j];
        s.vstage[slot] = val[j];
      }
    }

    uint32_t excl;
    if (single_wave) {
      // ---- one wave of tiles: every tile publishes its aggregate at about the same time, and a
      // chained walk would be ~tiles / 16 dependent L2 round trips.  Two-level sum instead: tiles
      // form groups of 2^gs_log (about sqrt(tiles)); the last tile of a group publishes the
      // group total as soon as it has read its group's aggregates; a tile adds the totals of the
      // earlier groups and the aggregates of the earlier tiles of its own group: three round
      // trips however many tiles there are.
      excl = s.digit_base[tid];
      const int g = tile >> gs_log, first = g << gs_log;
      uint32_t within = 0;
      for (int base = first; base < tile; base += LOOKBACK) {
        uint64_t w[LOOKBACK];
        bool ok;
        do {
          ok = true;
#pragma unroll
          for (int k = 0; k < LOOKBACK; ++k)
            w[k] = base + k < tile ? ld_volatile_u64(status + (size_t)(base + k) * RADIX + tid) : (ep | FLAG_AGG);
#pragma unroll
          for (int k = 0; k < LOOKBACK; ++k)
            if ((w[k] >> 32) != epoch || (w[k] & (FLAG_AGG | FLAG_INC)) == 0) ok = false;
        } while (!ok);
#pragma unroll
        for (int k = 0; k < LOOKBACK; ++k) within += (uint32_t)w[k] & VALUE_MASK;
      }
      if (tile == first + (1 << gs_log) - 1)
        st_volatile_u64(gstatus + (size_t)g * RADIX + tid, ep | FLAG_AGG | (within + count));
      excl += within;
      for (int base = 0; base < g; base += LOOKBACK) {
        uint64_t w[LOOKBACK];
        bool ok;
        do {
          ok = true;
#pragma unroll
          for (int k = 0; k < LOOKBACK; ++k)
            w[k] = base + k < g ? ld_volatile_u64(gstatus + (size_t)(base + k) * RADIX + tid) : (ep | FLAG_AGG);
#pragma unroll
          for (int k = 0; k < LOOKBACK; ++k)
            if ((w[k] >> 32) != epoch || (w[k] & FLAG_AGG) == 0) ok = false;
        } while (!ok);
#pragma unroll
        for (int k = 0; k < LOOKBACK; ++k) excl += (uint32_t)w[k] & VALUE_MASK;
      }
    } else
    {
    // ---- decoupled look-back for bin `tid`
    if (tile == 0) {
      excl = s.digit_base[tid];
    } else {
      excl = 0;
      // LOOKBACK predecessors per round trip: below a few million elements all tiles of a wave
      // publish their aggregates at about the same time, so the walk back to an inclusive
      // prefix is a chain of about tiles / (2 LOOKBACK) L2 round trips.
      int t = tile - 1;
      bool done = false;
      while (!done) {
        uint64_t w[LOOKBACK];
#pragma unroll
        for (int k = 0; k < LOOKBACK; ++k)
          w[k] = t - k >= 0 ? ld_volatile_u64(status + (size_t)(t - k) * RADIX + tid) : 0ull;
        bool stalled = false;
        int used = 0;
#pragma unroll
        for (int k = 0; k < LOOKBACK; ++k) {
          if (!done && !stalled) {
            if ((w[k] >> 32) != epoch || (w[k] & (FLAG_AGG | FLAG_INC)) == 0) {
              stalled = true;  // not published yet: poll again from this tile
            } else {
              excl += (uint32_t)w[k] & VALUE_MASK;
              ++used;
              if (w[k] & FLAG_INC) done = true;
            }
          }
        }
        t -= used;
      }
    }
    }
    if (!single_wave) st_volatile_u64(my, ep | FLAG_INC | (excl + count));
    s.bin_base[tid] = (int64_t)excl - (int64_t)toff;
    __syncthreads();

    // ---- out: runs of equal digits are contiguous in shared memory and in global memory
    const uint32_t tile_n = min((uint32_t)TILE, n - tile_base);
#pragma unroll
    for (int j = 0; j < ITEMS; ++j) {
      const uint32_t k = tid + j * SORT_THREADS;
      if (k < tile_n) {
        const uint64_t kk = s.stage[k];
        const int64_t pos = s.bin_base[(kk >> shift) & 0xff] + k;
        __stcg(kout + pos, kk);
        __stcg(vout + pos, s.vstage[k]);
      }
    }
    __syncthreads();
  }
}

// SORT_HYBRID, after the passes over bits 32..62: look for neighbours with equal top bits
// in this block's tiles.  The head of a run of 2..RUN_MAX elements sorts it in place (stable
// insertion sort by the full code; equal codes keep their order, which is id order); a longer
// run raises st->sort_fallback.
template <int ITEMS>
__device__ __forceinline__ void fixup_runs(uint64_t* key, uint32_t* val, FrameState* st, uint32_t n, int num_tiles, int low) {
  constexpr int TILE = SORT_THREADS * ITEMS;
  const int lane = threadIdx.x & 31;
  for (int tile = blockIdx.x; tile < num_tiles; tile += gridDim.x) {
    const uint32_t tile_base = (uint32_t)tile * TILE;
    // all keys of the thread first (ITEMS loads in flight); a lane's right neighbour is the next lane's key
    uint64_t k[ITEMS], kx[ITEMS];
#pragma unroll
    for (int j = 0; j < ITEMS; ++j) {
      const uint32_t idx = tile_base + j * SORT_THREADS + threadIdx.x;
      k[j] = idx < n ? __ldcg(key + idx) : 0ull;
      kx[j] = (lane == 31 && idx + 1 < n) ? __ldcg(key + idx + 1) : 0ull;
    }
#pragma unroll
    for (int j = 0; j < ITEMS; ++j) {
      const uint32_t idx = tile_base + j * SORT_THREADS + threadIdx.x;
      const uint64_t kd = __shfl_down_sync(0xffffffffu, k[j], 1);
      const uint64_t kn = lane == 31 ? kx[j] : kd;
      if (idx + 1 >= n || (k[j] >> low) != (kn >> low)) continue;   // common case: no run continues here
      if (idx > 0 && (__ldcg(key + idx - 1) >> low) == (k[j] >> low)) continue;  // not the head
      uint32_t len = 2;
      while (len <= RUN_MAX && idx + len < n && (__ldcg(key + idx + len) >> low) == (k[j] >> low)) ++len;
      if (len > RUN_MAX) {
        st->sort_fallback = 1u;
        continue;
      }
      for (uint32_t a = 1; a < len; ++a) {
        const uint64_t ka = __ldcg(key + idx + a);
        const uint32_t va = __ldcg(val + idx + a);
        uint32_t b = a;
        while (b > 0) {
          const uint64_t kb = __ldcg(key + idx + b - 1);
          if (!(kb > ka)) break;
          __stcg(key + idx + b, kb);
          __stcg(val + idx + b, __ldcg(val + idx + b - 1));
          --b;
        }
        if (b != a) {
          __stcg(key + idx + b, ka);
          __stcg(val + idx + b, va);
        }
      }
    }
  }
}

template <int ITEMS>
__device__ __forceinline__ void run_sort(SortSmem& s, const SortArgs& a, uint32_t n) {
  constexpr int TILE = SORT_THREADS * ITEMS;
  const int num_tiles = (int)((n + TILE - 1) / TILE);
  const uint32_t nb = min((uint32_t)gridDim.x, (uint32_t)num_tiles);  // blocks that own a tile
  if (blockIdx.x >= nb) return;
  uint32_t* bar = &a.st->sort_bar;
  uint32_t round = 0, epoch = a.epoch0;
  if (a.mode == SORT_SINGLE) {
    const int in = a.pass & 1;
    onesweep_pass<ITEMS>(s, a.key[in], a.val[in], a.key[in ^ 1], a.val[in ^ 1], a.st, a.pass, a.status, epoch, n, num_tiles);
    return;
  }
  int first = a.mode == SORT_HYBRID ? hybrid_first_digit(n) : 0;
  int buf = sort_input_buffer(a.mode, n);
  for (int pass = first;;) {
    onesweep_pass<ITEMS>(s, a.key[buf], a.val[buf], a.key[buf ^ 1], a.val[buf ^ 1], a.st, pass, a.status, epoch++, n, num_tiles);
    buf ^= 1;
    if (++pass < 8) {
      grid_barrier(bar, nb, round);
      continue;
    }
    if (first == 0) break;  // all 8 digits sorted
    grid_barrier(bar, nb, round);
    fixup_runs<ITEMS>(a.key[0], a.val[0], a.st, n, num_tiles, 8 * first);
    grid_barrier(bar, nb, round);
    if (*reinterpret_cast<volatile uint32_t*>(&a.st->sort_fallback) == 0u) break;
    // a long run of equal top bits: redo the sort with all 8 passes.  unproject_kernel counted only
    // the digits >= first, so count the low ones here (a histogram does not depend on the order).
    {
      const int tid = threadIdx.x;
      for (int d = 0; d < first; ++d) s.warp_hist[d][tid] = 0;
      __syncthreads();
      for (uint32_t idx = blockIdx.x * SORT_THREADS + tid; idx < n; idx += nb * SORT_THREADS) {
        const uint64_t k = __ldcg(a.key[0] + idx);
        for (int d = 0; d < first; ++d) atomicAdd(&s.warp_hist[d][(uint32_t)(k >> (8 * d)) & 0xff], 1u);
      }
      __syncthreads();
      for (int d = 0; d < first; ++d) {
        const uint32_t h = s.warp_hist[d][tid];
        if (h) atomicAdd(&a.st->hist[d][tid], h);
      }
      grid_barrier(bar, nb, round);
    }
    first = 0;
    pass = 0;
  }
}

// The tile size follows N (known on the device only).  One wave (every tile has a resident block):
// the smallest tile that still gives one wave -- small frames are latency bound, so they get the
// most blocks busy and the shortest ranking chains.  Several waves: the tile size that wastes the
// least of the last wave (cost model: waves x (items per thread + a fixed per-tile part)).
#ifndef SPLATS_SORT_BLOCKS
#define SPLATS_SORT_BLOCKS 2
#endif
#ifndef SPLATS_SORT_FIXED
#define SPLATS_SORT_FIXED 6
#endif
__device__ __forceinline__ int sort_pick_items(uint32_t n, uint32_t grid) {
  int best = SORT_MAX_ITEMS;
  uint32_t best_cost = 0xffffffffu;
  for (int items = 4; items <= SORT_MAX_ITEMS; items += 2) {
    const uint32_t tiles = (n + SORT_THREADS * items - 1) / (SORT_THREADS * items);
    if (tiles <= grid) return items;   // the smallest single-wave size
    const uint32_t cost = ((tiles + grid - 1) / grid) * (uint32_t)(items + SPLATS_SORT_FIXED);
    if (cost <= best_cost) { best_cost = cost; best = items; }
  }
  return best;
}
__global__ void __launch_bounds__(SORT_THREADS, SPLATS_SORT_BLOCKS)
onesweep_kernel(SortArgs a) {
  pdl_wait();
  pdl_trigger();
  extern __shared__ __align__(16) unsigned char smem_raw[];
  SortSmem& s = *reinterpret_cast<SortSmem*>(smem_raw);
  const uint32_t n = a.st->n;
  switch (sort_pick_items(n, gridDim.x)) {
    case 4: run_sort<4>(s, a, n); break;
    case 6: run_sort<6>(s, a, n); break;
    case 8: run_sort<8>(s, a, n); break;
#if SPLATS_SORT_MAX_ITEMS >= 16
    case 10: run_sort<10>(s, a, n); break;
    case 12: run_sort<12>(s, a, n); break;
    case 14: run_sort<14>(s, a, n); break;
    default: run_sort<16>(s, a, n); break;
#else
    default: run_sort<8>(s, a, n); break;
#endif
  }
}

}  // namespace sw
