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
constexpr int LOOKBACK = SPLATS_LOOKBACK;       // status words per round trip of the two-level sum (one wave)
#ifndef SPLATS_LOOKBACK_CHAIN
#define SPLATS_LOOKBACK_CHAIN 4
#endif
constexpr int LOOKBACK_CHAIN = SPLATS_LOOKBACK_CHAIN;   // ... of the chained look-back (several waves): measured 2 .. 8
constexpr int RUN_MAX = 32;           // longest run of equal top bits fixed up in place

struct SortArgs {
  uint64_t* key[2];
  uint32_t* val[2];
  FrameState* st;
  uint64_t* status;
  uint32_t epoch0;   // this launch may use epochs epoch0 .. epoch0 + 31
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
  uint64_t stage[SORT_THREADS * SORT_MAX_ITEMS];   // keys in tile-sorted order; window buffer A of the windowed sort
  uint32_t vstage[SORT_THREADS * SORT_MAX_ITEMS];  // values in tile-sorted order
  uint64_t stage2[SORT_THREADS * SORT_MAX_ITEMS];  // window buffer B
  uint32_t vstage2[SORT_THREADS * SORT_MAX_ITEMS];
  uint64_t mbar;                                    // mbarrier of the window phase's bulk copies
};
constexpr int WIN_MAX = SORT_THREADS * SORT_MAX_ITEMS;   // capacity of a window (4096 elements)

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

// Stable rank of one key per lane among the keys of the same digit that this warp has seen so far in the
// tile / window (warp_hist[warp] holds the running counts).
__device__ __forceinline__ uint32_t warp_rank(SortSmem& s, uint32_t dig, bool valid, int lane, int warp) {
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
  return base + before;
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
    for (int j = 0; j < ITEMS; ++j)
      rank[j] = warp_rank(s, (uint32_t)(key[j] >> shift) & 0xff, (wbase + j * 32) < n, lane, warp);
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
      // LOOKBACK_CHAIN predecessors per round trip: below a few million elements all tiles of a wave
      // publish their aggregates at about the same time, so the walk back to an inclusive
      // prefix is a chain of about tiles / (2 LOOKBACK_CHAIN) L2 round trips.
      int t = tile - 1;
      bool done = false;
      while (!done) {
        uint64_t w[LOOKBACK_CHAIN];
#pragma unroll
        for (int k = 0; k < LOOKBACK_CHAIN; ++k)
          w[k] = t - k >= 0 ? ld_volatile_u64(status + (size_t)(t - k) * RADIX + tid) : 0ull;
        bool stalled = false;
        int used = 0;
#pragma unroll
        for (int k = 0; k < LOOKBACK_CHAIN; ++k) {
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

// ---- windowed hybrid sort (SORT_HYBRID, the default): after three global passes over the top digits the
// array is a sequence of buckets of equal top 24 code bits (cells of 1/256 x 1/256 x 1/256 of the scene box: a
// few to a few hundred samples of a one-sample-per-pixel frame), in order; what is left is to put every bucket
// in order by (code, position): local work.  The array is cut into windows at bucket boundaries (window k =
// [B(k T), B((k + 1) T)), B(x) = first bucket start >= x); a block loads a window into shared memory, every
// thread takes an element and counts the keys of its bucket that come before it (stable, by the full code: no
// fix-up afterwards), which is its place, and the window is written back in place.  No status words, no look-back, no grid barrier.  A bucket that does not fit (> WIN_BUCKET_MAX keys, or
// a window > WIN_MAX) raises st->sort_wfall and the launch falls back to LSD passes.
#ifndef SPLATS_WIN_EXTRA
#define SPLATS_WIN_EXTRA 512
#endif
constexpr int WIN_BUCKET_MAX = SPLATS_WIN_EXTRA;      // counting is quadratic in the bucket size
static_assert(WIN_MAX <= (1 << 24), "comparison key = the key bits below the bucket's (<= 40) + position");

constexpr int WIN_EXTRA = SPLATS_WIN_EXTRA;           // a window is loaded with this many elements beyond its nominal end

// ---- bulk asynchronous copy global -> shared (cp.async.bulk, sm_90+): one thread asks the copy engine for a
// contiguous range; completion is counted in bytes on an mbarrier that every thread of the block waits on.
// Source, destination and size must be multiples of 16 bytes.
__device__ __forceinline__ uint32_t smem_addr(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" :: "r"(smem_addr(bar)), "r"(count) : "memory");
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" :: "r"(smem_addr(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
               :: "r"(smem_addr(dst)), "l"(src), "r"(bytes), "r"(smem_addr(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "WAIT_%=:\n\t"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
      "@!p bra WAIT_%=;\n\t}"
      :: "r"(smem_addr(bar)), "r"(parity) : "memory");
}

__device__ __forceinline__ void window_phase(SortSmem& s, uint64_t* key, uint32_t* val, FrameState* st, uint32_t n, const int WIN_BSHIFT) {
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  uint32_t* heads = s.tile_off;   // one bit per loaded element: a bucket starts here (128 words)
  // nominal window size: what the capacity allows, a quarter of it for small frames (more windows than blocks)
  const uint32_t T = n > (uint32_t)gridDim.x * (WIN_MAX / 4) ? WIN_MAX - WIN_EXTRA : WIN_MAX / 4;
  const uint32_t nwin = (n + T - 1) / T;
  if (tid == 0) mbar_init(&s.mbar, 1u);
  uint32_t phase = 0;
  __syncthreads();
  for (uint32_t k = blockIdx.x; k < nwin; k += gridDim.x) {
    // ---- load [k T, (k + 1) T + WIN_EXTRA) in one go; the window proper, [B(k T), B((k + 1) T)), is found in it.
    // The loaded range overlaps the neighbouring windows, which other blocks may be writing at the same time.
    // That is harmless: outside its own window a block looks at the bucket bits of a key only (to find the heads),
    // and a neighbour only permutes keys inside buckets, so those bits are the same before, during and after its
    // writes (64-bit stores: a key is seen old or new, never torn); the windows proper are disjoint.
    // Keys and values come as two bulk asynchronous copies (up to 32 + 16 KiB; g0 is a multiple of 4 elements, so
    // both ranges are 16-byte aligned); the up to three elements behind the last multiple of four are loaded by hand.
    const uint32_t g0 = k * T, gend = min(n, g0 + T + WIN_EXTRA), cnt = gend - g0, cnt4 = cnt & ~3u;
    if (tid == 0 && cnt4) {
      // the staging buffers were read and written through the generic proxy (previous window, earlier passes), the
      // global arrays by other blocks before the grid barrier: order all of that before the async proxy's accesses
      asm volatile("fence.proxy.async;" ::: "memory");
      mbar_expect_tx(&s.mbar, cnt4 * 12u);
      bulk_g2s(s.stage, key + g0, cnt4 * 8u, &s.mbar);
      bulk_g2s(s.vstage, val + g0, cnt4 * 4u, &s.mbar);
    }
    if (tid < (int)(cnt - cnt4)) {
      s.stage[cnt4 + tid] = __ldcg(key + g0 + cnt4 + tid);
      s.vstage[cnt4 + tid] = __ldcg(val + g0 + cnt4 + tid);
    }
    const uint64_t kprev = g0 > 0 ? __ldcg(key + g0 - 1) : 0ull;
    if (cnt4) {
      mbar_wait(&s.mbar, phase);
      phase ^= 1u;
    }
    __syncthreads();
    // bucket heads as a bit map (chunk c = elements 32 c .. 32 c + 31 of the loaded range)
    const uint32_t nchunk = (cnt + 31) >> 5;
    for (uint32_t c = warp; c < nchunk; c += SORT_WARPS) {
      const uint32_t i = c * 32 + lane;
      const bool head = i < cnt && ((i == 0 && g0 == 0) || ((i == 0 ? kprev : s.stage[i - 1]) >> WIN_BSHIFT) != (s.stage[i] >> WIN_BSHIFT));
      const unsigned m = __ballot_sync(0xffffffffu, head);
      if (lane == 0) heads[c] = m;
      // comparison key inside a bucket: the 39 code bits below the bucket's, then the position (unique: no ties)
      if (i < cnt) s.stage2[i] = (s.stage[i] << (64 - WIN_BSHIFT)) | i;
    }
    __syncthreads();
    // first head >= x in the loaded range, cnt if none
    auto first_head = [&](uint32_t x) -> uint32_t {
      uint32_t c = x >> 5;
      if (c >= nchunk) return cnt;
      uint32_t w = heads[c] & (0xffffffffu << (x & 31));
      while (!w) {
        if (++c >= nchunk) return cnt;
        w = heads[c];
      }
      return c * 32 + (uint32_t)__ffs(w) - 1u;
    };
    const uint32_t w0 = first_head(0);                                        // B(k T) - g0
    const uint32_t w1 = g0 + T >= n ? cnt : first_head(T);                    // B((k + 1) T) - g0
    if ((w0 == cnt && g0 + cnt < n) || (w1 == cnt && g0 + cnt < n)) {         // no boundary within WIN_EXTRA: a bucket too large
      if (tid == 0) st->sort_wfall = 1u;
      __syncthreads();
      continue;
    }
    // one thread per element of the window: its bucket [p, q) from the bit map, its place = p + the number of keys
    // of the bucket that come before it (smaller code, or the same code and an earlier position: stable)
    for (uint32_t i = w0 + tid; i < w1; i += SORT_THREADS) {
      int c = (int)(i >> 5);
      uint32_t w = heads[c] & (0xffffffffu >> (31 - (i & 31)));   // heads at or before i in its chunk
      while (!w) w = heads[--c];                                     // w0 is a head
      const uint32_t p = (uint32_t)c * 32 + 31u - (uint32_t)__clz(w);
      const uint32_t q = min(first_head(i + 1), w1);
      if (q - p > WIN_BUCKET_MAX) {   // counting is quadratic: leave the bucket as it is and fall back
        st->sort_wfall = 1u;
        continue;
      }
      const uint64_t ti = s.stage2[i];
      uint32_t rank = 0;
#pragma unroll 4
      for (uint32_t j = p; j < q; ++j) rank += s.stage2[j] < ti ? 1u : 0u;
      __stcg(key + g0 + p + rank, s.stage[i]);   // everything is read from shared memory: writing in place is safe
      __stcg(val + g0 + p + rank, s.vstage[i]);
    }
    __syncthreads();
  }
}

// digit histograms that unproject_kernel did not count (digits lo .. hi - 1), from the keys in `key`
__device__ __noinline__ void count_digits(SortSmem& s, const uint64_t* key, FrameState* st, uint32_t n, uint32_t nb, int lo, int hi) {
  const int tid = threadIdx.x;
  if (lo >= hi) return;
  for (int d = lo; d < hi; ++d) s.warp_hist[d][tid] = 0;
  __syncthreads();
  for (uint32_t idx = blockIdx.x * SORT_THREADS + tid; idx < n; idx += nb * SORT_THREADS) {
    const uint64_t k = __ldcg(key + idx);
    for (int d = lo; d < hi; ++d) atomicAdd(&s.warp_hist[d][(uint32_t)(k >> (8 * d)) & 0xff], 1u);
  }
  __syncthreads();
  for (int d = lo; d < hi; ++d) {
    const uint32_t h = s.warp_hist[d][tid];
    if (h) atomicAdd(&st->hist[d][tid], h);
  }
}

// LSD passes over the digits from .. 7 (inlined at its three call sites: as a real call it costs 2 % of the sort)
template <int ITEMS>
__device__ __forceinline__ void lsd_passes(SortSmem& s, const SortArgs& a, uint32_t n, int num_tiles, uint32_t nb, int from, int& buf,
                                        uint32_t& epoch, uint32_t& round) {
  for (int pass = from; pass < 8; ++pass) {
    if (blockIdx.x < nb)
      onesweep_pass<ITEMS>(s, a.key[buf], a.val[buf], a.key[buf ^ 1], a.val[buf ^ 1], a.st, pass, a.status, epoch, n, num_tiles);
    ++epoch;
    buf ^= 1;
    grid_barrier(&a.st->sort_bar, gridDim.x, round);
  }
}

template <int ITEMS>
__device__ __forceinline__ void run_sort(SortSmem& s, const SortArgs& a, uint32_t n) {
  constexpr int TILE = SORT_THREADS * ITEMS;
  const int num_tiles = (int)((n + TILE - 1) / TILE);
  const uint32_t nb = min((uint32_t)gridDim.x, (uint32_t)num_tiles);  // blocks that own a tile
  uint32_t* bar = &a.st->sort_bar;
  uint32_t round = 0, epoch = a.epoch0;
  if (a.mode == SORT_SINGLE) {
    if (blockIdx.x >= nb) return;
    const int in = a.pass & 1;
    onesweep_pass<ITEMS>(s, a.key[in], a.val[in], a.key[in ^ 1], a.val[in ^ 1], a.st, a.pass, a.status, epoch, n, num_tiles);
    return;
  }
  // LSD passes over the digits from .. 7, buffer `buf` -> ... ; a grid barrier after every pass
  auto lsd = [&](int from, int& buf) { lsd_passes<ITEMS>(s, a, n, num_tiles, nb, from, buf, epoch, round); };
  int first = sort_is_hybrid(a.mode) ? hybrid_first_digit(n) : 0;
  int buf = sort_input_buffer(a.mode, n);
  if (a.mode == SORT_HYBRID) {
    // ---- three global passes over the top digits, then bucket by bucket in shared memory
    const int WIN_G = win_passes(n);
    lsd(8 - WIN_G, buf);                 // ends in buffer 0 (sort_input_buffer)
    window_phase(s, a.key[0], a.val[0], a.st, n, 8 * (8 - WIN_G));
    grid_barrier(bar, gridDim.x, round);
    if (*reinterpret_cast<volatile uint32_t*>(&a.st->sort_wfall) == 0u) return;
    // a bucket did not fit: LSD passes over the digits d0 .. 7 from where the array is now (every step so far
    // was a stable permutation; d0 is even so that the result ends in buffer 0), then the global fix-up
    const int d0 = first & ~1;
    count_digits(s, a.key[0], a.st, n, gridDim.x, d0, 8 - WIN_G);   // unproject_kernel counted the digits of the global passes only
    grid_barrier(bar, gridDim.x, round);
    lsd(d0, buf);
    if (blockIdx.x < nb) fixup_runs<ITEMS>(a.key[0], a.val[0], a.st, n, num_tiles, 8 * first);
    grid_barrier(bar, gridDim.x, round);
    first = d0;
    if (*reinterpret_cast<volatile uint32_t*>(&a.st->sort_fallback) == 0u) return;
  } else {
    lsd(first, buf);
    if (first == 0) return;  // all 8 digits sorted
    if (blockIdx.x < nb) fixup_runs<ITEMS>(a.key[0], a.val[0], a.st, n, num_tiles, 8 * first);
    grid_barrier(bar, gridDim.x, round);
    if (*reinterpret_cast<volatile uint32_t*>(&a.st->sort_fallback) == 0u) return;
  }
  // a long run of equal sorted bits: redo the sort with all 8 passes.  unproject_kernel counted only the digits
  // >= first, so count the low ones here (a histogram does not depend on the order).
  count_digits(s, a.key[0], a.st, n, gridDim.x, 0, first);
  grid_barrier(bar, gridDim.x, round);
  buf = 0;
  lsd(0, buf);
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
#if !SPLATS_LATE_TRIGGER
  pdl_trigger();   // (with SPLATS_LATE_TRIGGER the dependent launch is released when the blocks exit)
#endif
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
