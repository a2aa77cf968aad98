// splats_api.cu -- host side of the C ABI declared in include/splats.h: one context that owns
// all device memory, argument checks, and the kernel launch sequence of the two hot calls.
// Nothing here computes on the CPU except the per-call camera constants; there is no CPU
// fallback (every entry point fails with SPLATS_ECUDA / SPLATS_ESTATE without a device).
#include "../../include/splats.h"

#include <algorithm>
#include <cmath>
#include <cstddef>
#include <cstdio>
#include <cstring>
#include <string>
#include <vector>

#include "build_kernels.cuh"
#include "common.cuh"
#include "lbvh.cuh"
#include "march.cuh"
#include "onesweep.cuh"
#include "pack.cuh"
#include "points.cuh"
#include "render.cuh"
#include "tree_tile.cuh"

#ifndef SPLATS_PDL_MASK
#define SPLATS_PDL_MASK 63
#endif

namespace {

using namespace sw;

constexpr int SORT_MIN_TILE = SORT_THREADS * 4;  // smallest tile of onesweep_kernel
static_assert(SPLATS_SORT_HYBRID == SORT_HYBRID && SPLATS_SORT_LSD8 == SORT_LSD8 && SPLATS_SORT_LSD8_LAUNCHES == SORT_SINGLE &&
              SPLATS_SORT_HYBRID_LSD == SORT_HYBRID_LSD,
              "public sort modes must match onesweep.cuh");

struct Context {
  cudaStream_t stream = nullptr;
  int max_w = 0, max_h = 0;
  int64_t cap = 0;
  int num_sms = 0;
  // device memory
  FrameState* state = nullptr;      // [3]: frame f uses state[f % 3] and re-arms state[(f + 1) % 3]
  uint32_t* tile_count = nullptr;   // [cap / TILE_PX + 1]
  uint32_t* pack_tile_count = nullptr;  // the same for splats_pack, which may run while a build is in flight
  unsigned* sched = nullptr;        // render tile ticket + done counter, one pair per render in flight
  unsigned long long* traced = nullptr;   // pixels for which the renders set up a ray (splats_traced_pixels)
  // renders launched since the last fully serialising launch on the stream (see do_render)
  static constexpr int MAX_OVERLAP = 8;
  int render_streak = 0;
  bool last_was_render = false;         // the last thing enqueued on the stream by this library is a render launched with PDL
  bool serialize_next_render = false;   // set when renders may be in flight that the bookkeeping below no longer knows
  const char* inflight_lo[MAX_OVERLAP] = {};
  const char* inflight_hi[MAX_OVERLAP] = {};
  uint64_t* key[2] = {nullptr, nullptr};
  uint32_t* val[2] = {nullptr, nullptr};
  uint64_t* status = nullptr;       // [max sort tiles][256]
  size_t status_bytes = 0;
  // Two complete BVHs: build f writes set[f & 1] while the renders may still read the other one
  // (splats_update_begin / splats_update_commit); splats, colours, ids, nodes in sorted order.
  struct BvhSet {
    float4* sphere = nullptr;
    float4* rgba = nullptr;
    uint32_t* ids = nullptr;
    QNode* qnodes = nullptr;    // 32-byte traversal records, always written
    Node* nodes = nullptr;      // exact 64-byte records: written by the pyramid / atomic refit modes, and by the
                                // tiled mode only while SPLATS_OPT_EXACT_NODES is on
    bool has_exact = false;     // `nodes` holds the exact records of this set's current BVH
  } set[2];
  int cur_set = 0, cur_state = 0;   // what splats_render* reads
  // a build enqueued by splats_update_begin that splats_update_commit has not made current yet
  bool pending = false;
  int pending_set = 0, pending_state = 0;
  cudaStream_t build_stream = nullptr;   // high priority; created on the first splats_update_begin
  cudaEvent_t ev_begin = nullptr, ev_built = nullptr;
  uint64_t* zkey = nullptr;         // depth buffer of splats_render_points, all ones between calls
  int* leaf_parent = nullptr;
  float4* pyr = nullptr;            // min/max pyramid over the leaf boxes (lbvh.cuh), 2 float4 per entry
  int4* ranges = nullptr;           // (first, split, last) of every internal node, hierarchy_kernel -> boxes_kernel; tiled mode: the queue of tree_spine_kernel
  float4* sphere_px = nullptr;      // splat (centre, radius) of every valid source pixel, bounds_kernel -> unproject_kernel, tree gather
  uint8_t* tile_min = nullptr;      // tiled tree: smallest delta + 1 of every tile of sorted leaves
  uint16_t* tile_fb = nullptr;      // tiled tree: first / last split below every threshold, per tile
  PyramidLayout pyr_layout;
  int refit_mode = SPLATS_REFIT_TILED;
  int sort_mode = SPLATS_SORT_HYBRID;
  int radius_mode = SPLATS_RADIUS_FOOTPRINT;
  bool pdl = true;                  // programmatic dependent launches between the hot-path kernels
  bool exact_nodes = false;         // SPLATS_OPT_EXACT_NODES
  bool overlap = false;             // consecutive independent renders may run concurrently (SPLATS_OPT_OVERLAP)
  float radius_param = 0.0f;
  // staging for the *_host calls: copies run on their own streams, double / triple buffered,
  // so the upload of frame f+1 and the read-back of image i-1 overlap the kernels of image i
  static constexpr int N_IN = 2, N_OUT = 3;
  cudaStream_t h2d_stream = nullptr, d2h_stream = nullptr;
  float* stage_color[N_IN] = {nullptr, nullptr};
  float* stage_depth[N_IN] = {nullptr, nullptr};
  float* stage_out[N_OUT] = {nullptr, nullptr, nullptr};
  cudaEvent_t in_uploaded[N_IN] = {}, in_free[N_IN] = {};    // h2d done / kernels done reading
  cudaEvent_t out_rendered[N_OUT] = {}, out_free[N_OUT] = {};  // render done / d2h done
  unsigned n_uploads = 0, n_readbacks = 0;
  // frame bookkeeping
  unsigned frame = 0;               // number of updates enqueued
  uint32_t epoch = 0;
  bool has_bvh = false;
  int sort_grid = 0;
  int render_grid = 0;
  size_t sort_smem = 0;
  // profiling
  bool profiling = false;
  std::vector<cudaEvent_t> pool;    // events, grown on demand while profiling is on
  size_t pool_used = 0;
  struct Span { int stage; size_t e0, e1; };
  std::vector<Span> spans;          // one per (call, stage) since the last splats_stage_ms
  unsigned long long launches = 0;

  size_t mark() {                   // record the next pooled event on the stream
    if (pool_used == pool.size()) {
      cudaEvent_t e = nullptr;
      cudaEventCreate(&e);
      pool.push_back(e);
    }
    cudaEventRecord(pool[pool_used], stream);
    return pool_used++;
  }
};

Context* g_ctx = nullptr;
std::string g_err = "";

int fail(int code, const std::string& msg) {
  g_err = msg;
  return code;
}

int cuda_fail(cudaError_t e, const char* what) {
  return fail(SPLATS_ECUDA, std::string(what) + ": " + cudaGetErrorString(e));
}

#define CU(call)                                   \
  do {                                             \
    cudaError_t e_ = (call);                       \
    if (e_ != cudaSuccess) return cuda_fail(e_, #call); \
  } while (0)

bool finite_camera(const wr_camera* c) {
  const float* f = reinterpret_cast<const float*>(c);
  for (int i = 0; i < 13; ++i)
    if (!std::isfinite(f[i])) return false;
  return c->tan_half_fovy > 0.0f;
}

DevCamera make_camera(const wr_camera* c, int W, int H) {
  DevCamera d;
  for (int k = 0; k < 3; ++k) { d.e[k] = c->eye[k]; d.R[k] = c->right[k]; d.U[k] = c->up[k]; d.F[k] = c->fwd[k]; }
  d.tau = c->tan_half_fovy;
  d.fW = (float)W;
  d.fH = (float)H;
  volatile float tw = d.tau * d.fW;  // two separately rounded float32 operations
  d.ta = tw / d.fH;
  d.W = W;
  d.H = H;
  return d;
}

// k_r = r_scale * sqrt(1/2) * (2 tau / H), each product / quotient rounded to float32.
float radius_factor(const wr_camera* c, int H, float r_scale) {
  const float SQRT_HALF = 0.70710678118654752440f;
  volatile float a = r_scale * SQRT_HALF;
  volatile float b = 2.0f * c->tan_half_fovy;
  volatile float q = b / (float)H;
  return a * q;
}

// Launch on the context's stream, optionally as a programmatic dependent launch (common.cuh).
template <typename... KArgs, typename... Args>
void launch(bool pdl, void (*kernel)(KArgs...), int grid, int block, size_t smem, cudaStream_t s, Args... args) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3((unsigned)grid);
  cfg.blockDim = dim3((unsigned)block);
  cfg.dynamicSmemBytes = smem;
  cfg.stream = s;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = pdl ? 1 : 0;
  cudaLaunchKernelEx(&cfg, kernel, static_cast<KArgs>(args)...);
}

template <typename T>
cudaError_t dmalloc(T** p, size_t count) {
  return cudaMalloc(reinterpret_cast<void**>(p), count * sizeof(T));
}

void free_all(Context* c) {
  cudaFree(c->state); cudaFree(c->tile_count); cudaFree(c->pack_tile_count); cudaFree(c->sched); cudaFree(c->traced);
  cudaFree(c->key[0]); cudaFree(c->key[1]); cudaFree(c->val[0]); cudaFree(c->val[1]);
  cudaFree(c->status);
  for (int i = 0; i < 2; ++i) { cudaFree(c->set[i].sphere); cudaFree(c->set[i].rgba); cudaFree(c->set[i].ids); cudaFree(c->set[i].qnodes); cudaFree(c->set[i].nodes); }
  if (c->build_stream) cudaStreamDestroy(c->build_stream);
  if (c->ev_begin) cudaEventDestroy(c->ev_begin);
  if (c->ev_built) cudaEventDestroy(c->ev_built);
  cudaFree(c->leaf_parent); cudaFree(c->pyr); cudaFree(c->ranges); cudaFree(c->zkey); cudaFree(c->tile_min); cudaFree(c->sphere_px); cudaFree(c->tile_fb);
  for (int i = 0; i < Context::N_IN; ++i) {
    cudaFree(c->stage_color[i]); cudaFree(c->stage_depth[i]);
    if (c->in_uploaded[i]) cudaEventDestroy(c->in_uploaded[i]);
    if (c->in_free[i]) cudaEventDestroy(c->in_free[i]);
  }
  for (int i = 0; i < Context::N_OUT; ++i) {
    cudaFree(c->stage_out[i]);
    if (c->out_rendered[i]) cudaEventDestroy(c->out_rendered[i]);
    if (c->out_free[i]) cudaEventDestroy(c->out_free[i]);
  }
  if (c->h2d_stream) cudaStreamDestroy(c->h2d_stream);
  if (c->d2h_stream) cudaStreamDestroy(c->d2h_stream);
  for (auto& e : c->pool)
    if (e) cudaEventDestroy(e);
}

int ensure_staging(Context* c) {
  if (!c->h2d_stream) {
    CU(cudaStreamCreateWithFlags(&c->h2d_stream, cudaStreamNonBlocking));
    CU(cudaStreamCreateWithFlags(&c->d2h_stream, cudaStreamNonBlocking));
    for (int i = 0; i < Context::N_IN; ++i) {
      CU(dmalloc(&c->stage_color[i], (size_t)c->cap * 4));
      CU(dmalloc(&c->stage_depth[i], (size_t)c->cap));
      CU(cudaEventCreateWithFlags(&c->in_uploaded[i], cudaEventDisableTiming));
      CU(cudaEventCreateWithFlags(&c->in_free[i], cudaEventDisableTiming));
    }
    for (int i = 0; i < Context::N_OUT; ++i) {
      CU(dmalloc(&c->stage_out[i], (size_t)c->cap * 4));
      CU(cudaEventCreateWithFlags(&c->out_rendered[i], cudaEventDisableTiming));
      CU(cudaEventCreateWithFlags(&c->out_free[i], cudaEventDisableTiming));
    }
  }
  return SPLATS_OK;
}

// Quantisation constants of the wire format, each operation rounded to float32 on its own.
bool make_quant(const wr_quant* q, QuantParams* out) {
  for (int k = 0; k < 3; ++k) {
    if (!std::isfinite(q->lo[k]) || !std::isfinite(q->hi[k]) || !(q->hi[k] > q->lo[k])) return false;
    volatile float ext = q->hi[k] - q->lo[k];
    volatile float cell = ext / 65536.0f;
    if (!std::isfinite(ext)) return false;
    out->lo[k] = q->lo[k];
    out->ext[k] = ext;
    out->cell[k] = cell;
  }
  if (!(q->r_max > 0.0f) || !std::isfinite(q->r_max)) return false;
  volatile float rstep = q->r_max / 65535.0f;
  out->r_max = q->r_max;
  out->rstep = rstep;
  return true;
}

RadiusParams make_radius(const Context* c, const wr_camera* cam, int H, float r_scale) {
  RadiusParams rp;
  rp.mode = c->radius_mode;
  rp.k_r = radius_factor(cam, H, r_scale);
  volatile float rc = r_scale * c->radius_param;   // separately rounded float32 operations
  volatile float w1 = 1.0f - c->radius_param;
  rp.r_const = rc;
  rp.f_min = c->radius_param;
  rp.w1 = w1;
  return rp;
}

// ---- splats_pack_noalloc (include/splats.h): the compaction's per-tile counts in a file-scope device array
// instead of context memory.  One word per tile of TILE_PX pixels; 32 KiB + one line, resident on every GPU that
// loads this library until the process exits.  In host code the NAME of the array is a host-side stand-in, not
// a device address: the kernels get the address that cudaGetSymbolAddress returns for the current device.
constexpr int NOALLOC_MAX_TILES = SPLATS_NOALLOC_MAX_PIXELS / TILE_PX;
static __device__ __align__(256) uint32_t g_noalloc_tile_count[NOALLOC_MAX_TILES + 64];

constexpr int NOALLOC_MAX_DEVICES = 64;
struct NoallocDevice {
  uint32_t* tile_count = nullptr;   // device address of g_noalloc_tile_count on this device
  int num_sms = 0;
};
NoallocDevice g_noalloc[NOALLOC_MAX_DEVICES];

// Once per device, with that device current.  No allocation: a symbol look-up and an attribute query.
int noalloc_device(NoallocDevice** out) {
  int dev = 0;
  CU(cudaGetDevice(&dev));
  if (dev < 0 || dev >= NOALLOC_MAX_DEVICES) return fail(SPLATS_EINVAL, "splats_pack_noalloc: device index beyond 63");
  NoallocDevice& d = g_noalloc[dev];
  if (!d.tile_count) {
    uint32_t* ptr = nullptr;
    cudaError_t e = cudaGetSymbolAddress(reinterpret_cast<void**>(&ptr), g_noalloc_tile_count);
    if (e != cudaSuccess) return cuda_fail(e, "cudaGetSymbolAddress(g_noalloc_tile_count)");
    if (!ptr) return fail(SPLATS_ECUDA, "cudaGetSymbolAddress returned a null address for the static scratch array");
    int sms = 0;
    CU(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    d.num_sms = sms;
    d.tile_count = ptr;
  }
  *out = &d;
  return SPLATS_OK;
}

// The launch sequence of one update: a1 bounds, a2 keys + compaction, a3 sort, a4/a5 tree.
// Src yields the splat centres of elements [0, P) (build_kernels.cuh), Gather the sphere and
// colour of a splat id (lbvh.cuh).
template <class Src, class Gather>
int do_update(Context* c, const Src& src, const Gather& gather, int64_t P, bool async = false) {
  if (c->pending) return fail(SPLATS_ESTATE, "a build started by splats_update_begin is pending: call splats_update_commit first");
  // build f goes to BVH set f & 1 and frame state f % 3 and re-arms state (f + 1) % 3; both were
  // last used by build f - 2 whose renders are complete (stream order, or the begin/commit protocol)
  const int tset = (int)(c->frame & 1u), tstate = (int)(c->frame % 3u);
  FrameState* st = c->state + tstate;
  FrameState* st_next = c->state + (tstate + 1) % 3;
  Context::BvhSet& bs = c->set[tset];
  const int tiles = P > 0 ? (int)((P + TILE_PX - 1) / TILE_PX) : 1;
  cudaStream_t s = async ? c->build_stream : c->stream;
  const bool prof = c->profiling && !async;   // per-stage events live on the caller's stream

  size_t m[6] = {0, 0, 0, 0, 0, 0};
  if (prof) m[0] = c->mark();
  const bool pdl = c->pdl && !prof;   // per-stage events need the stages to be disjoint in time
  // Which kernels are launched as programmatic dependents (SPLATS_OPT_PDL): bounds (1), unproject (2), sort (4),
  // tile (8), spine (16), the first render after an update (32).  Measured per kernel; with the early release of
  // the dependents only behind short kernels (common.cuh, SPLATS_LATE_TRIGGER) all of them gain: dense update
  // 0.291 -> 0.283 ms, config 3 11.0 k -> 11.2 k frames/s against 35 (sort, tile and spine as ordinary launches).
  constexpr int pdl_mask = SPLATS_PDL_MASK;
  if (!async) c->render_streak = 0;   // (a decoupled build runs on its own stream: the renders in flight stay tracked)
  // bounds_kernel waits for its predecessor at its first instruction; overlapping renders
  // complete in launch order (render.cuh), so everything before it in the stream is complete
  // after a render launched by this library (and nothing else since) the bounds kernel may start under its tail
  const int bounds_wait = (pdl && c->overlap && !async && c->last_was_render) ? 0 : 1;
  c->last_was_render = false;
  launch(pdl && (pdl_mask & 1), bounds_kernel<Src>, tiles, BUILD_THREADS, 0, s, src, P, st, c->tile_count, bounds_wait);
  if (prof) m[1] = c->mark();
  const int grid2 = tiles < c->num_sms * 8 ? tiles : c->num_sms * 8;
  launch(pdl && (pdl_mask & 2), unproject_kernel<Src>, grid2, BUILD_THREADS, 0, s, src, P, tiles, st, st_next, c->tile_count, c->key[0],
         c->val[0], c->key[1], c->val[1], c->sort_mode);
  if (prof) m[2] = c->mark();
  const int max_sort_tiles = P > 0 ? (int)((P + SORT_MIN_TILE - 1) / SORT_MIN_TILE) : 1;
  const int sgrid = max_sort_tiles < c->sort_grid ? max_sort_tiles : c->sort_grid;
  if (c->epoch > 0xffffff00u) {   // the look-back words carry a 32-bit epoch: start over with a clean array before it wraps
    cudaMemsetAsync(c->status, 0, c->status_bytes, s);
    c->epoch = 0;
  }
  SortArgs sa;
  sa.key[0] = c->key[0]; sa.key[1] = c->key[1];
  sa.val[0] = c->val[0]; sa.val[1] = c->val[1];
  sa.st = st;
  sa.status = c->status;
  sa.mode = c->sort_mode;
  int sort_launches = 1;
  if (c->sort_mode == SORT_SINGLE) {
    sort_launches = 8;
    for (int pass = 0; pass < 8; ++pass) {
      sa.pass = pass;
      sa.epoch0 = ++c->epoch;
      onesweep_kernel<<<sgrid, SORT_THREADS, c->sort_smem, s>>>(sa);
    }
  } else {
    sa.pass = 0;
    sa.epoch0 = c->epoch + 1;
    c->epoch += 32;
    launch(pdl && (pdl_mask & 4), onesweep_kernel, sgrid, SORT_THREADS, c->sort_smem, s, sa);
  }
  if (prof) m[3] = c->mark();
  const int lgrid_max = P > 0 ? (int)((P + LBVH_THREADS - 1) / LBVH_THREADS) : 1;
  const int lgrid = lgrid_max < c->num_sms * 8 ? lgrid_max : c->num_sms * 8;
  if (c->refit_mode == SPLATS_REFIT_ATOMIC) {
    emit_kernel<Gather><<<lgrid, LBVH_THREADS, 0, s>>>(c->key[0], c->val[0], gather, st, bs.sphere, bs.rgba, bs.ids, bs.nodes,
                                                       c->leaf_parent);
    if (prof) m[4] = c->mark();
    refit_kernel<<<lgrid, LBVH_THREADS, 0, s>>>(bs.sphere, c->leaf_parent, bs.nodes, st);
    quantise_nodes_kernel<<<lgrid, LBVH_THREADS, 0, s>>>((const Node*)bs.nodes, (const FrameState*)st, bs.qnodes);
    c->launches += 1;
    bs.has_exact = true;
  } else if (c->refit_mode == SPLATS_REFIT_TILED) {
    // gather + leaf boxes + pyramid + every node whose range lies inside one tile of sorted leaves;
    // then the few nodes that span tiles (lbvh.cuh)
    const int tgrid = P > 0 ? (int)((P + TT_LEAVES - 1) / TT_LEAVES) : 1;
    launch(pdl && (pdl_mask & 8), tree_tile_kernel<Gather>, tgrid, TT_THREADS, sizeof(TileSmem), s, (const uint64_t*)c->key[0], (const uint32_t*)c->val[0],
           gather, st, bs.sphere, bs.rgba, bs.ids, reinterpret_cast<uint4*>(c->pyr), bs.qnodes, c->ranges, c->tile_min, c->tile_fb);
    if (prof) m[4] = c->mark();
    int nt_log = 0;
    while ((1 << nt_log) < tgrid) ++nt_log;
    const int sgrid2 = std::min(c->num_sms * 8, (tgrid * TT_QMAX + 7) / 8);   // persistent, one warp per queued node; idle blocks exit at once
    launch(pdl && (pdl_mask & 16), tree_spine_kernel, sgrid2, SPINE_THREADS, (size_t)2 << nt_log, s, (const uint64_t*)c->key[0], st, (const int4*)c->ranges,
           (const float4*)bs.sphere, (const uint4*)c->pyr, bs.qnodes, (const uint8_t*)c->tile_min, (const uint16_t*)c->tile_fb, nt_log);
    bs.has_exact = false;
    if (c->exact_nodes) {
      // SPLATS_OPT_EXACT_NODES: the tiled build carries quantised boxes only, so the exact float32 records (parity
      // tests, splats_export) come from the pyramid refit run after it on the same sorted keys: Karras' per-node
      // searches and exact range unions.  It rewrites sphere / rgba / ids with the same values and leaves qnodes alone.
      const int pgrid = P > 0 ? (int)((P + PYR_LEAVES - 1) / PYR_LEAVES) : 1;
      leaf_pyramid_kernel<Gather><<<pgrid, PYR_THREADS, 0, s>>>(c->val[0], gather, st, bs.sphere, bs.rgba, bs.ids, c->pyr);
      hierarchy_kernel<<<lgrid, LBVH_THREADS, 0, s>>>((const uint64_t*)c->key[0], (const FrameState*)st, c->ranges, 1);
      boxes_kernel<<<lgrid, LBVH_THREADS, 0, s>>>((const int4*)c->ranges, (const float4*)bs.sphere, (const float4*)c->pyr, st, bs.nodes);
      c->launches += 3;
      bs.has_exact = true;
    }
  } else {
    const int pgrid = P > 0 ? (int)((P + PYR_LEAVES - 1) / PYR_LEAVES) : 1;
    launch(pdl, leaf_pyramid_kernel<Gather>, pgrid, PYR_THREADS, 0, s, c->val[0], gather, st, bs.sphere, bs.rgba, bs.ids, c->pyr);
    if (prof) m[4] = c->mark();
    // the hierarchy (keys only) runs beside the pyramid (ids only); boxes_kernel joins them
    launch(pdl, hierarchy_kernel, lgrid, LBVH_THREADS, 0, s, (const uint64_t*)c->key[0], (const FrameState*)st, c->ranges, pdl ? 0 : 1);
    launch(pdl, boxes_kernel, lgrid, LBVH_THREADS, 0, s, (const int4*)c->ranges, (const float4*)bs.sphere, (const float4*)c->pyr, st, bs.nodes);
    launch(pdl, quantise_nodes_kernel, lgrid, LBVH_THREADS, 0, s, (const Node*)bs.nodes, (const FrameState*)st, bs.qnodes);
    c->launches += 2;
    bs.has_exact = true;
  }
  if (prof) m[5] = c->mark();
  c->launches += 4 + sort_launches;
  if (prof)
    for (int i = 0; i < 5; ++i) c->spans.push_back({i, m[i], m[i + 1]});
  CU(cudaGetLastError());
  c->frame += 1;
  if (async) {
    c->pending = true;
    c->pending_set = tset;
    c->pending_state = tstate;
  } else {
    c->cur_set = tset;
    c->cur_state = tstate;
    c->has_bvh = true;
  }
  return SPLATS_OK;
}

int do_update_frame(Context* c, const float* color, const float* depth, const wr_camera* cam, int W, int H, float r_scale,
                    bool async = false) {
  FrameSource src;
  src.depth = depth;
  src.color = reinterpret_cast<const float4*>(color);
  src.sphere_px = c->sphere_px;
  src.cam = make_camera(cam, W, H);
  src.rp = make_radius(c, cam, H, r_scale);
  FrameGather g;
  g.sphere_px = c->sphere_px;
  g.color = src.color;
  return do_update(c, src, g, (int64_t)W * H, async);
}

int do_render(Context* c, const wr_camera* cam, int W2, int H2, float* out, bool first_hit = false, bool rgba8 = false) {
  RenderParams prm;
  prm.cam = make_camera(cam, W2, H2);
  prm.qnodes = c->set[c->cur_set].qnodes;
  prm.sphere = c->set[c->cur_set].sphere;
  prm.rgba = c->set[c->cur_set].rgba;
  prm.ids = c->set[c->cur_set].ids;
  prm.st = c->state + c->cur_state;
  prm.out = reinterpret_cast<float4*>(out);
  prm.out8 = reinterpret_cast<uint32_t*>(out);
  prm.traced = c->traced;
  const int tiles = ((W2 + 7) / 8) * ((H2 + 3) / 4);
  const int blocks_needed = (tiles + RENDER_THREADS / 32 - 1) / (RENDER_THREADS / 32);
  const int grid = blocks_needed < c->render_grid ? blocks_needed : c->render_grid;  // persistent (render.cuh)
  size_t m0 = 0;
  if (c->profiling) m0 = c->mark();
  // Renders of one BVH into disjoint images do not depend on each other, so up to MAX_OVERLAP
  // consecutive ones are launched as programmatic dependents that do NOT wait for their
  // predecessor: the next render's blocks fill the SMs that the tail of the previous one leaves
  // idle.  The first render after anything else waits (the BVH must be complete; everything
  // before it in the stream is ordered), every MAX_OVERLAP-th one and any render whose image
  // overlaps one that may still be in flight is an ordinary launch (full stream order).  A
  // render that skips the wait at its start waits at its end (render.cuh), so renders complete
  // in launch order and whatever follows is ordered after all of them.  Each render in flight
  // has its own pair of ticket counters.
  const char* out_lo = reinterpret_cast<const char*>(out);
  const char* out_hi = out_lo + (size_t)W2 * H2 * (rgba8 ? 4 : 16);
  bool pdl = c->pdl && !c->profiling;
  int wait_prev = 1;
  if (c->serialize_next_render) {   // e.g. after splats_update_commit: earlier renders may still be running
    pdl = false;
    c->render_streak = 0;
    c->serialize_next_render = false;
  } else if (!(pdl && c->overlap)) {
    c->render_streak = 0;   // every render waits for its predecessor; one pair of ticket counters
  } else if (c->render_streak > 0) {
    bool independent = c->render_streak < Context::MAX_OVERLAP;
    for (int i = 0; i < c->render_streak && independent; ++i)
      if (out_lo < c->inflight_hi[i] && c->inflight_lo[i] < out_hi) independent = false;
    if (independent) {
      wait_prev = 0;
    } else {
      pdl = false;          // an ordinary launch: serialised against everything before it
      c->render_streak = 0;
    }
  }
  prm.wait_prev = wait_prev;
  prm.sched = c->sched + 2 * c->render_streak;
  c->inflight_lo[c->render_streak] = out_lo;
  c->inflight_hi[c->render_streak] = out_hi;
  c->render_streak = (pdl && c->overlap) ? c->render_streak + 1 : 0;
  constexpr int pdl_mask = SPLATS_PDL_MASK;
  const bool attr = pdl && (wait_prev == 0 || (pdl_mask & 32));
  if (rgba8) launch(attr, render_kernel<KBUF, false, true>, grid, RENDER_THREADS, 0, c->stream, prm);
  else if (first_hit) launch(attr, render_kernel<1, true, false>, grid, RENDER_THREADS, 0, c->stream, prm);
  else launch(attr, render_kernel<KBUF, false, false>, grid, RENDER_THREADS, 0, c->stream, prm);
  if (c->profiling) c->spans.push_back({5, m0, c->mark()});
  c->last_was_render = pdl;
  c->launches += 1;
  CU(cudaGetLastError());
  return SPLATS_OK;
}

int check_frame_args(Context* c, const void* a, const void* b, const wr_camera* cam, int W, int H) {
  if (!c) return fail(SPLATS_ESTATE, "no context: call splats_create first");
  if (!a || !b || !cam) return fail(SPLATS_EINVAL, "null pointer argument");
  if (W <= 0 || H <= 0 || (int64_t)W * H > c->cap) return fail(SPLATS_EINVAL, "W*H outside [1, capacity]");
  if (!finite_camera(cam)) return fail(SPLATS_EINVAL, "camera is not finite or tan_half_fovy <= 0");
  return SPLATS_OK;
}

}  // namespace

extern "C" {

int splats_create(void* cuda_stream, int max_W, int max_H) {
  if (g_ctx) return fail(SPLATS_ESTATE, "context already exists: call splats_destroy first");
  if (max_W <= 0 || max_H <= 0 || (int64_t)max_W * max_H >= (1ll << 26))
    return fail(SPLATS_EINVAL, "max_W*max_H outside [1, 2^26)");
  int dev = 0;
  CU(cudaGetDevice(&dev));
  Context* c = new Context();
  c->stream = reinterpret_cast<cudaStream_t>(cuda_stream);
  c->max_w = max_W;
  c->max_h = max_H;
  c->cap = (int64_t)max_W * max_H;
  cudaError_t e = cudaDeviceGetAttribute(&c->num_sms, cudaDevAttrMultiProcessorCount, dev);
  const size_t cap = (size_t)c->cap;
  const size_t max_sort_tiles = (cap + SORT_MIN_TILE - 1) / SORT_MIN_TILE;
  if (e == cudaSuccess) e = dmalloc(&c->state, 3);
  if (e == cudaSuccess) e = dmalloc(&c->tile_count, cap / TILE_PX + 2);
  if (e == cudaSuccess) e = dmalloc(&c->pack_tile_count, cap / TILE_PX + 2);
  if (e == cudaSuccess) e = dmalloc(&c->sched, 2 * Context::MAX_OVERLAP);
  if (e == cudaSuccess) e = cudaMemset(c->sched, 0, 2 * Context::MAX_OVERLAP * sizeof(unsigned));
  if (e == cudaSuccess) e = dmalloc(&c->traced, 1);
  if (e == cudaSuccess) e = cudaMemset(c->traced, 0, sizeof(unsigned long long));
  for (int i = 0; i < 2 && e == cudaSuccess; ++i) {
    e = dmalloc(&c->key[i], cap);
    if (e == cudaSuccess) e = dmalloc(&c->val[i], cap);
  }
  const size_t status_rows = max_sort_tiles + max_sort_tiles / 8 + 4;   // tile words + group totals (onesweep.cuh)
  if (e == cudaSuccess) e = dmalloc(&c->status, status_rows * RADIX);
  for (int i = 0; i < 2 && e == cudaSuccess; ++i) {
    e = dmalloc(&c->set[i].sphere, cap);
    if (e == cudaSuccess) e = dmalloc(&c->set[i].rgba, cap);
    if (e == cudaSuccess) e = dmalloc(&c->set[i].ids, cap);
    if (e == cudaSuccess) e = dmalloc(&c->set[i].qnodes, cap);
    if (e == cudaSuccess) e = dmalloc(&c->set[i].nodes, cap);
  }
  if (e == cudaSuccess) e = dmalloc(&c->leaf_parent, cap);
  if (e == cudaSuccess) e = dmalloc(&c->ranges, cap);
  if (e == cudaSuccess) e = dmalloc(&c->tile_min, cap / TT_LEAVES + 2);
  if (e == cudaSuccess) e = dmalloc(&c->sphere_px, cap);
  if (e == cudaSuccess) e = dmalloc(&c->tile_fb, (cap / TT_LEAVES + 2) * 2 * TT_VPAD);
  if (e == cudaSuccess) e = dmalloc(&c->zkey, cap);
  if (e == cudaSuccess) e = cudaMemset(c->zkey, 0xff, cap * sizeof(uint64_t));
  {  // pyramid levels 1.. : ceil(cap / 2^k) entries each
    size_t off = 0;
    c->pyr_layout.off[0] = 0;
    for (int k = 1; k <= PYR_MAX_LEVELS; ++k) {
      c->pyr_layout.off[k] = (uint32_t)off;
      off += (cap + ((size_t)1 << k) - 1) >> k;
    }
    if (e == cudaSuccess) e = dmalloc(&c->pyr, 2 * off);
    if (e == cudaSuccess) e = cudaMemcpyToSymbol(c_pyr, &c->pyr_layout, sizeof(PyramidLayout));
  }
  c->status_bytes = status_rows * RADIX * sizeof(uint64_t);
  if (e == cudaSuccess) e = cudaMemset(c->status, 0, c->status_bytes);
  if (e == cudaSuccess) {
    FrameState init;
    memset(&init, 0, sizeof(init));
    for (int a = 0; a < 3; ++a) init.lo[a] = 0xffffffffu;
    for (int i = 0; i < 3 && e == cudaSuccess; ++i)
      e = cudaMemcpy(c->state + i, &init, sizeof(init), cudaMemcpyHostToDevice);
  }
  if (e == cudaSuccess) e = cudaFuncSetAttribute(tree_spine_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 160 * 1024);
  if (e == cudaSuccess) e = cudaFuncSetAttribute(tree_tile_kernel<FrameGather>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(TileSmem));
  if (e == cudaSuccess) e = cudaFuncSetAttribute(tree_tile_kernel<PackedGather>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(TileSmem));
  if (e == cudaSuccess) {
    c->sort_smem = sizeof(SortSmem);
    e = cudaFuncSetAttribute(onesweep_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c->sort_smem);
  }
  int occ = 0;
  if (e == cudaSuccess)
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, onesweep_kernel, SORT_THREADS, c->sort_smem);
  if (e == cudaSuccess && occ < 1) { free_all(c); delete c; return fail(SPLATS_ECUDA, "onesweep kernel does not fit on an SM"); }
  if (e != cudaSuccess) {
    free_all(c);
    delete c;
    return cuda_fail(e, "splats_create");
  }
  c->sort_grid = c->num_sms * occ;  // co-resident persistent grid (see onesweep.cuh)
  int rocc = 0;
  e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&rocc, render_kernel<KBUF, false>, RENDER_THREADS, 0);
  if (e != cudaSuccess || rocc < 1) {
    free_all(c);
    delete c;
    return e != cudaSuccess ? cuda_fail(e, "splats_create") : fail(SPLATS_ECUDA, "render kernel does not fit on an SM");
  }
  c->render_grid = c->num_sms * rocc;
  g_ctx = c;
  return SPLATS_OK;
}

int splats_update(const float* color, const float* depth, const wr_camera* src_camera, int W, int H, float r_scale) {
  int rc = check_frame_args(g_ctx, color, depth, src_camera, W, H);
  if (rc) return rc;
  if (!(r_scale > 0.0f) || !std::isfinite(r_scale)) return fail(SPLATS_EINVAL, "r_scale must be finite and > 0");
  if ((reinterpret_cast<uintptr_t>(color) | reinterpret_cast<uintptr_t>(depth)) & 15u)
    return fail(SPLATS_EINVAL, "color/depth must be 16-byte aligned");
  return do_update_frame(g_ctx, color, depth, src_camera, W, H, r_scale);
}

// Start of a decoupled build: everything enqueued so far on the caller's stream happens before
// it, nothing enqueued later waits for it until splats_update_commit.
int begin_build(Context* c) {
  if (c->pending) return fail(SPLATS_ESTATE, "a build started by splats_update_begin is already pending");
  if (!c->build_stream) {
    int lo = 0, hi = 0;
    CU(cudaDeviceGetStreamPriorityRange(&lo, &hi));   // hi = numerically lowest = highest priority
    CU(cudaStreamCreateWithPriority(&c->build_stream, cudaStreamNonBlocking, hi));
    CU(cudaEventCreateWithFlags(&c->ev_begin, cudaEventDisableTiming));
    CU(cudaEventCreateWithFlags(&c->ev_built, cudaEventDisableTiming));
  }
  CU(cudaEventRecord(c->ev_begin, c->stream));
  CU(cudaStreamWaitEvent(c->build_stream, c->ev_begin, 0));
  return SPLATS_OK;
}

int splats_update_begin(const float* color, const float* depth, const wr_camera* src_camera, int W, int H, float r_scale) {
  int rc = check_frame_args(g_ctx, color, depth, src_camera, W, H);
  if (rc) return rc;
  if (!(r_scale > 0.0f) || !std::isfinite(r_scale)) return fail(SPLATS_EINVAL, "r_scale must be finite and > 0");
  if ((reinterpret_cast<uintptr_t>(color) | reinterpret_cast<uintptr_t>(depth)) & 15u)
    return fail(SPLATS_EINVAL, "color/depth must be 16-byte aligned");
  rc = begin_build(g_ctx);
  if (rc) return rc;
  rc = do_update_frame(g_ctx, color, depth, src_camera, W, H, r_scale, true);
  if (rc) return rc;
  CU(cudaEventRecord(g_ctx->ev_built, g_ctx->build_stream));
  return SPLATS_OK;
}

int splats_update_commit(void) {
  if (!g_ctx) return fail(SPLATS_ESTATE, "no context: call splats_create first");
  Context* c = g_ctx;
  if (!c->pending) return fail(SPLATS_ESTATE, "splats_update_commit without splats_update_begin");
  CU(cudaStreamWaitEvent(c->stream, c->ev_built, 0));
  c->cur_set = c->pending_set;
  c->cur_state = c->pending_state;
  c->pending = false;
  c->has_bvh = true;
  c->serialize_next_render = true;   // the renders of the previous BVH may still be in flight
  return SPLATS_OK;
}

int splats_render(const wr_camera* dst_camera, int W2, int H2, float* out_rgba) {
  int rc = check_frame_args(g_ctx, out_rgba, out_rgba, dst_camera, W2, H2);
  if (rc) return rc;
  if (reinterpret_cast<uintptr_t>(out_rgba) & 15u) return fail(SPLATS_EINVAL, "out_rgba must be 16-byte aligned");
  if (!g_ctx->has_bvh) return fail(SPLATS_ENOBVH, "splats_render before any splats_update");
  return do_render(g_ctx, dst_camera, W2, H2, out_rgba);
}

int splats_render_first_hit(const wr_camera* dst_camera, int W2, int H2, float* out_rgba) {
  int rc = check_frame_args(g_ctx, out_rgba, out_rgba, dst_camera, W2, H2);
  if (rc) return rc;
  if (reinterpret_cast<uintptr_t>(out_rgba) & 15u) return fail(SPLATS_EINVAL, "out_rgba must be 16-byte aligned");
  if (!g_ctx->has_bvh) return fail(SPLATS_ENOBVH, "splats_render_first_hit before any splats_update");
  return do_render(g_ctx, dst_camera, W2, H2, out_rgba, true);
}

int splats_render_points(const wr_camera* dst_camera, int W2, int H2, int point_px, float* out_rgba) {
  int rc = check_frame_args(g_ctx, out_rgba, out_rgba, dst_camera, W2, H2);
  if (rc) return rc;
  if (reinterpret_cast<uintptr_t>(out_rgba) & 15u) return fail(SPLATS_EINVAL, "out_rgba must be 16-byte aligned");
  if (point_px < 1 || point_px > 64) return fail(SPLATS_EINVAL, "point_px outside [1, 64]");
  Context* c = g_ctx;
  if (!c->has_bvh) return fail(SPLATS_ENOBVH, "splats_render_points before any update");
  PointParams p;
  p.cam = make_camera(dst_camera, W2, H2);
  p.sphere = c->set[c->cur_set].sphere;
  p.rgba = c->set[c->cur_set].rgba;
  p.ids = c->set[c->cur_set].ids;
  p.st = c->state + c->cur_state;
  p.zkey = c->zkey;
  p.out = reinterpret_cast<float4*>(out_rgba);
  p.point_px = point_px;
  p.hW = 0.5f * (float)W2;
  p.hH = 0.5f * (float)H2;
  p.off = 0.5f * (float)point_px + 0.5f;
  const int grid = c->num_sms * 8;
  size_t m0 = 0;
  if (c->profiling) m0 = c->mark();
  c->render_streak = 0;
  c->last_was_render = false;
  points_kernel<false><<<grid, POINT_THREADS, 0, c->stream>>>(p);
  points_kernel<true><<<grid, POINT_THREADS, 0, c->stream>>>(p);
  points_background_kernel<<<grid, POINT_THREADS, 0, c->stream>>>(p);
  if (c->profiling) c->spans.push_back({7, m0, c->mark()});
  c->launches += 3;
  CU(cudaGetLastError());
  return SPLATS_OK;
}

int splats_march(const float* volume, int n, const wr_transfer* tf, const wr_camera* camera, int W, int H, float* color,
                 float* depth) {
  int rc = check_frame_args(g_ctx, color, depth, camera, W, H);
  if (rc) return rc;
  if (!volume || !tf) return fail(SPLATS_EINVAL, "null pointer argument");
  if (n < 1 || n > 2048) return fail(SPLATS_EINVAL, "volume size outside [1, 2048]");
  if (tf->n_tents < 1 || tf->n_tents > 4) return fail(SPLATS_EINVAL, "n_tents outside [1, 4]");
  if (!(tf->half_width > 0.0f) || !std::isfinite(tf->half_width)) return fail(SPLATS_EINVAL, "half_width must be finite and > 0");
  if (reinterpret_cast<uintptr_t>(color) & 15u) return fail(SPLATS_EINVAL, "color must be 16-byte aligned");
  Context* c = g_ctx;
  MarchParams p;
  p.vol = volume;
  p.n = n;
  p.fn = (float)n;
  volatile float step = 0.5f / p.fn;
  p.step = step;
  p.n_tents = tf->n_tents;
  for (int i = 0; i < 4; ++i) {
    p.iso[i] = tf->iso[i];
    p.amax[i] = tf->alpha[i];
    for (int k = 0; k < 3; ++k) p.rgb[i][k] = tf->rgb[i][k];
  }
  p.hw = tf->half_width;
  p.shade = tf->shade;
  volatile float oms = 1.0f - tf->shade;
  p.one_minus_shade = oms;
  p.depth_alpha = tf->depth_alpha;
  p.stop_alpha = tf->stop_alpha;
  p.cam = make_camera(camera, W, H);
  p.color = reinterpret_cast<float4*>(color);
  p.depth = depth;
  const int tiles = ((W + 7) / 8) * ((H + 3) / 4);
  const int blocks_needed = (tiles + MARCH_THREADS / 32 - 1) / (MARCH_THREADS / 32);
  const int grid = blocks_needed < c->num_sms * 16 ? blocks_needed : c->num_sms * 16;
  size_t m0 = 0;
  if (c->profiling) m0 = c->mark();
  c->render_streak = 0;
  c->last_was_render = false;
  march_kernel<<<grid, MARCH_THREADS, 0, c->stream>>>(p);
  if (c->profiling) c->spans.push_back({8, m0, c->mark()});
  c->launches += 1;
  CU(cudaGetLastError());
  return SPLATS_OK;
}

int splats_pack(const float* color, const float* depth, const wr_camera* src_camera, int W, int H, float r_scale,
                const wr_quant* quant, unsigned long long* samples, unsigned* colors, unsigned* count) {
  int rc = check_frame_args(g_ctx, color, depth, src_camera, W, H);
  if (rc) return rc;
  if (!quant || !samples || !colors || !count) return fail(SPLATS_EINVAL, "null pointer argument");
  if (!(r_scale > 0.0f) || !std::isfinite(r_scale)) return fail(SPLATS_EINVAL, "r_scale must be finite and > 0");
  if ((reinterpret_cast<uintptr_t>(color) | reinterpret_cast<uintptr_t>(depth)) & 15u)
    return fail(SPLATS_EINVAL, "color/depth must be 16-byte aligned");
  Context* c = g_ctx;
  PackArgs a;
  if (!make_quant(quant, &a.q)) return fail(SPLATS_EINVAL, "quantisation box must be finite with hi > lo, r_max finite and > 0");
  a.color = reinterpret_cast<const float4*>(color);
  a.depth = depth;
  a.cam = make_camera(src_camera, W, H);
  a.rp = make_radius(c, src_camera, H, r_scale);
  a.P = (int64_t)W * H;
  a.num_tiles = (int)((a.P + TILE_PX - 1) / TILE_PX);
  size_t m0 = 0;
  if (c->profiling) m0 = c->mark();
  c->render_streak = 0;
  c->last_was_render = false;
  pack_count_kernel<<<a.num_tiles, BUILD_THREADS, 0, c->stream>>>(a, c->pack_tile_count);
  const int grid2 = a.num_tiles < c->num_sms * 4 ? a.num_tiles : c->num_sms * 4;
  pack_write_kernel<<<grid2, BUILD_THREADS, 0, c->stream>>>(a, c->pack_tile_count, reinterpret_cast<uint64_t*>(samples), colors, count);
  if (c->profiling) c->spans.push_back({6, m0, c->mark()});
  c->launches += 2;
  CU(cudaGetLastError());
  return SPLATS_OK;
}

int splats_noalloc_setup(void) {
  NoallocDevice* d = nullptr;
  return noalloc_device(&d);
}

int splats_pack_noalloc(const float* color, const float* depth, const wr_camera* src_camera, int W, int H, float r_scale,
                        int radius_mode, float radius_param, const wr_quant* quant, unsigned long long* samples,
                        unsigned* colors, unsigned* count, void* cuda_stream) {
  // needs no context and calls no cudaMalloc / cudaFree: everything it touches is the caller's or the static array
  if (!color || !depth || !src_camera || !quant || !samples || !colors || !count) return fail(SPLATS_EINVAL, "null pointer argument");
  if (W <= 0 || H <= 0) return fail(SPLATS_EINVAL, "W and H must be positive");
  if ((int64_t)W * H > (int64_t)SPLATS_NOALLOC_MAX_PIXELS)
    return fail(SPLATS_EINVAL, "splats_pack_noalloc: W*H = " + std::to_string((long long)W * H) + " exceeds the static scratch array's maximum of " +
                                   std::to_string((long long)SPLATS_NOALLOC_MAX_PIXELS) + " pixels (SPLATS_NOALLOC_MAX_PIXELS); use splats_pack");
  if (!finite_camera(src_camera)) return fail(SPLATS_EINVAL, "camera is not finite or tan_half_fovy <= 0");
  if (!(r_scale > 0.0f) || !std::isfinite(r_scale)) return fail(SPLATS_EINVAL, "r_scale must be finite and > 0");
  if ((reinterpret_cast<uintptr_t>(color) | reinterpret_cast<uintptr_t>(depth)) & 15u)
    return fail(SPLATS_EINVAL, "color/depth must be 16-byte aligned");
  if (radius_mode != SPLATS_RADIUS_FOOTPRINT && radius_mode != SPLATS_RADIUS_CONSTANT && radius_mode != SPLATS_RADIUS_OPACITY)
    return fail(SPLATS_EINVAL, "unknown radius mode");
  if (radius_mode == SPLATS_RADIUS_CONSTANT && !(radius_param > 0.0f && std::isfinite(radius_param)))
    return fail(SPLATS_EINVAL, "constant radius must be finite and > 0");
  if (radius_mode == SPLATS_RADIUS_OPACITY && !(radius_param >= 0.0f && radius_param <= 1.0f))
    return fail(SPLATS_EINVAL, "opacity radius floor must be in [0, 1]");
  PackArgs a;
  if (!make_quant(quant, &a.q)) return fail(SPLATS_EINVAL, "quantisation box must be finite with hi > lo, r_max finite and > 0");
  NoallocDevice* d = nullptr;
  int rc = noalloc_device(&d);
  if (rc) return rc;
  a.color = reinterpret_cast<const float4*>(color);
  a.depth = depth;
  a.cam = make_camera(src_camera, W, H);
  {  // as make_radius, with the mode and parameter of the call (separately rounded float32 operations)
    const float param = radius_mode == SPLATS_RADIUS_FOOTPRINT ? 0.0f : radius_param;
    a.rp.mode = radius_mode;
    a.rp.k_r = radius_factor(src_camera, H, r_scale);
    volatile float rc_ = r_scale * param;
    volatile float w1 = 1.0f - param;
    a.rp.r_const = rc_;
    a.rp.f_min = param;
    a.rp.w1 = w1;
  }
  a.P = (int64_t)W * H;
  a.num_tiles = (int)((a.P + TILE_PX - 1) / TILE_PX);   // <= NOALLOC_MAX_TILES by the check above
  cudaStream_t s = reinterpret_cast<cudaStream_t>(cuda_stream);
  // the array keeps the previous call's counts; pack_count_kernel overwrites every word [0, num_tiles) that
  // pack_write_kernel reads, so nothing has to be cleared
  pack_count_kernel<<<a.num_tiles, BUILD_THREADS, 0, s>>>(a, d->tile_count);
  const int grid2 = a.num_tiles < d->num_sms * 4 ? a.num_tiles : d->num_sms * 4;
  pack_write_kernel<<<grid2, BUILD_THREADS, 0, s>>>(a, d->tile_count, reinterpret_cast<uint64_t*>(samples), colors, count);
  CU(cudaGetLastError());
  return SPLATS_OK;
}

int splats_update_packed(const unsigned long long* samples, const unsigned* colors, unsigned n, const wr_quant* quant) {
  if (!g_ctx) return fail(SPLATS_ESTATE, "no context: call splats_create first");
  if (!quant || ((!samples || !colors) && n != 0)) return fail(SPLATS_EINVAL, "null pointer argument");
  if ((int64_t)n > g_ctx->cap) return fail(SPLATS_EINVAL, "n exceeds the capacity given to splats_create");
  if (reinterpret_cast<uintptr_t>(samples) & 15u) return fail(SPLATS_EINVAL, "samples must be 16-byte aligned");
  PackedSource src;
  if (!make_quant(quant, &src.q)) return fail(SPLATS_EINVAL, "quantisation box must be finite with hi > lo, r_max finite and > 0");
  src.samples = reinterpret_cast<const uint64_t*>(samples);
  PackedGather g;
  g.samples = src.samples;
  g.colours = colors;
  g.q = src.q;
  return do_update(g_ctx, src, g, (int64_t)n);
}

int splats_update_packed_host(const unsigned long long* samples_host, const unsigned* colors_host, unsigned n,
                              const wr_quant* quant) {
  if (!g_ctx) return fail(SPLATS_ESTATE, "no context: call splats_create first");
  if (!quant || ((!samples_host || !colors_host) && n != 0)) return fail(SPLATS_EINVAL, "null pointer argument");
  if ((int64_t)n > g_ctx->cap) return fail(SPLATS_EINVAL, "n exceeds the capacity given to splats_create");
  Context* c = g_ctx;
  PackedSource src;
  if (!make_quant(quant, &src.q)) return fail(SPLATS_EINVAL, "quantisation box must be finite with hi > lo, r_max finite and > 0");
  int rc = ensure_staging(c);
  if (rc) return rc;
  // the frame staging buffers are reused: 16 bytes per pixel hold the 8-byte samples, 4 the colours
  const int u = (int)(c->n_uploads % Context::N_IN);
  if (c->n_uploads >= (unsigned)Context::N_IN) CU(cudaStreamWaitEvent(c->h2d_stream, c->in_free[u], 0));
  if (n) {
    CU(cudaMemcpyAsync(c->stage_color[u], samples_host, (size_t)n * sizeof(uint64_t), cudaMemcpyHostToDevice, c->h2d_stream));
    CU(cudaMemcpyAsync(c->stage_depth[u], colors_host, (size_t)n * sizeof(uint32_t), cudaMemcpyHostToDevice, c->h2d_stream));
  }
  CU(cudaEventRecord(c->in_uploaded[u], c->h2d_stream));
  CU(cudaStreamWaitEvent(c->stream, c->in_uploaded[u], 0));
  c->last_was_render = false;
  src.samples = reinterpret_cast<const uint64_t*>(c->stage_color[u]);
  PackedGather g;
  g.samples = src.samples;
  g.colours = reinterpret_cast<const uint32_t*>(c->stage_depth[u]);
  g.q = src.q;
  rc = do_update(c, src, g, (int64_t)n);
  if (rc) return rc;
  CU(cudaEventRecord(c->in_free[u], c->stream));
  c->n_uploads += 1;
  return SPLATS_OK;
}

int splats_update_host(const float* color_host, const float* depth_host, const wr_camera* src_camera, int W, int H,
                       float r_scale) {
  int rc = check_frame_args(g_ctx, color_host, depth_host, src_camera, W, H);
  if (rc) return rc;
  if (!(r_scale > 0.0f) || !std::isfinite(r_scale)) return fail(SPLATS_EINVAL, "r_scale must be finite and > 0");
  Context* c = g_ctx;
  rc = ensure_staging(c);
  if (rc) return rc;
  const size_t P = (size_t)W * H;
  const int u = (int)(c->n_uploads % Context::N_IN);
  if (c->n_uploads >= (unsigned)Context::N_IN) CU(cudaStreamWaitEvent(c->h2d_stream, c->in_free[u], 0));
  CU(cudaMemcpyAsync(c->stage_color[u], color_host, P * 4 * sizeof(float), cudaMemcpyHostToDevice, c->h2d_stream));
  CU(cudaMemcpyAsync(c->stage_depth[u], depth_host, P * sizeof(float), cudaMemcpyHostToDevice, c->h2d_stream));
  CU(cudaEventRecord(c->in_uploaded[u], c->h2d_stream));
  CU(cudaStreamWaitEvent(c->stream, c->in_uploaded[u], 0));
  c->last_was_render = false;
  rc = do_update_frame(c, c->stage_color[u], c->stage_depth[u], src_camera, W, H, r_scale);
  if (rc) return rc;
  CU(cudaEventRecord(c->in_free[u], c->stream));
  c->n_uploads += 1;
  return SPLATS_OK;
}

int splats_render_host(const wr_camera* dst_camera, int W2, int H2, float* out_rgba_host) {
  int rc = check_frame_args(g_ctx, out_rgba_host, out_rgba_host, dst_camera, W2, H2);
  if (rc) return rc;
  Context* c = g_ctx;
  if (!c->has_bvh) return fail(SPLATS_ENOBVH, "splats_render_host before any update");
  rc = ensure_staging(c);
  if (rc) return rc;
  const int r = (int)(c->n_readbacks % Context::N_OUT);
  if (c->n_readbacks >= (unsigned)Context::N_OUT) CU(cudaStreamWaitEvent(c->stream, c->out_free[r], 0));
  c->last_was_render = false;
  rc = do_render(c, dst_camera, W2, H2, c->stage_out[r]);
  if (rc) return rc;
  CU(cudaEventRecord(c->out_rendered[r], c->stream));
  c->last_was_render = false;   // an event record follows the render in the stream
  CU(cudaStreamWaitEvent(c->d2h_stream, c->out_rendered[r], 0));
  CU(cudaMemcpyAsync(out_rgba_host, c->stage_out[r], (size_t)W2 * H2 * 4 * sizeof(float), cudaMemcpyDeviceToHost,
                     c->d2h_stream));
  CU(cudaEventRecord(c->out_free[r], c->d2h_stream));
  c->n_readbacks += 1;
  return SPLATS_OK;
}

int splats_render_rgba8(const wr_camera* dst_camera, int W2, int H2, unsigned* out_rgba8) {
  int rc = check_frame_args(g_ctx, out_rgba8, out_rgba8, dst_camera, W2, H2);
  if (rc) return rc;
  if (reinterpret_cast<uintptr_t>(out_rgba8) & 3u) return fail(SPLATS_EINVAL, "out_rgba8 must be 4-byte aligned");
  if (!g_ctx->has_bvh) return fail(SPLATS_ENOBVH, "splats_render_rgba8 before any update");
  return do_render(g_ctx, dst_camera, W2, H2, reinterpret_cast<float*>(out_rgba8), false, true);
}

int splats_render_host_rgba8(const wr_camera* dst_camera, int W2, int H2, unsigned* out_rgba8_host) {
  int rc = check_frame_args(g_ctx, out_rgba8_host, out_rgba8_host, dst_camera, W2, H2);
  if (rc) return rc;
  Context* c = g_ctx;
  if (!c->has_bvh) return fail(SPLATS_ENOBVH, "splats_render_host_rgba8 before any update");
  rc = ensure_staging(c);
  if (rc) return rc;
  const int r = (int)(c->n_readbacks % Context::N_OUT);
  if (c->n_readbacks >= (unsigned)Context::N_OUT) CU(cudaStreamWaitEvent(c->stream, c->out_free[r], 0));
  c->last_was_render = false;
  rc = do_render(c, dst_camera, W2, H2, c->stage_out[r], false, true);
  if (rc) return rc;
  CU(cudaEventRecord(c->out_rendered[r], c->stream));
  c->last_was_render = false;   // an event record follows the render in the stream
  CU(cudaStreamWaitEvent(c->d2h_stream, c->out_rendered[r], 0));
  CU(cudaMemcpyAsync(out_rgba8_host, c->stage_out[r], (size_t)W2 * H2 * sizeof(unsigned), cudaMemcpyDeviceToHost, c->d2h_stream));
  CU(cudaEventRecord(c->out_free[r], c->d2h_stream));
  c->n_readbacks += 1;
  return SPLATS_OK;
}

int splats_count(unsigned* n_host) {
  if (!g_ctx) return fail(SPLATS_ESTATE, "no context");
  if (!n_host) return fail(SPLATS_EINVAL, "null pointer argument");
  Context* c = g_ctx;
  if (!c->has_bvh) { *n_host = 0; return SPLATS_OK; }
  CU(cudaMemcpyAsync(n_host, &c->state[c->cur_state].n, sizeof(unsigned), cudaMemcpyDeviceToHost, c->stream));
  CU(cudaStreamSynchronize(c->stream));
  return SPLATS_OK;
}

int splats_export(unsigned long long* keys, unsigned* perm, int* children, int* parents, float* node_aabbs) {
  if (!g_ctx) return fail(SPLATS_ESTATE, "no context");
  Context* c = g_ctx;
  if (!c->has_bvh) return fail(SPLATS_ENOBVH, "splats_export before any update");
  if (c->pending) return fail(SPLATS_ESTATE, "splats_export while a build is pending (its sorted keys are scratch of the build)");
  unsigned n = 0;
  int rc = splats_count(&n);
  if (rc) return rc;
  if (n == 0) return SPLATS_OK;
  if (keys) {
    export_keys_kernel<<<(int)((n + LBVH_THREADS - 1) / LBVH_THREADS), LBVH_THREADS, 0, c->stream>>>(
        (const uint64_t*)c->key[0], (const FrameState*)(c->state + c->cur_state), reinterpret_cast<uint64_t*>(keys));
    c->launches += 1;
  }
  if (perm) CU(cudaMemcpyAsync(perm, c->set[c->cur_set].ids, (size_t)n * sizeof(uint32_t), cudaMemcpyDeviceToDevice, c->stream));
  if (node_aabbs && !c->set[c->cur_set].has_exact)
    return fail(SPLATS_ESTATE, "splats_export: the exact node boxes were not stored by the last build (set SPLATS_OPT_EXACT_NODES before the update)");
  if (children || parents || node_aabbs) {
    if (parents) CU(cudaMemsetAsync(parents, 0xff, (size_t)(2 * n - 1) * sizeof(int), c->stream));
    const int grid = (int)((n + LBVH_THREADS - 1) / LBVH_THREADS);
    export_kernel<<<grid, LBVH_THREADS, 0, c->stream>>>(c->set[c->cur_set].qnodes, c->set[c->cur_set].nodes, c->set[c->cur_set].sphere, c->state + c->cur_state, children, parents,
                                                        node_aabbs);
    c->launches += 1;
    CU(cudaGetLastError());
  }
  CU(cudaStreamSynchronize(c->stream));
  return SPLATS_OK;
}

int splats_export_child_boxes(float* child_boxes) {
  if (!g_ctx) return fail(SPLATS_ESTATE, "no context");
  Context* c = g_ctx;
  if (!child_boxes) return fail(SPLATS_EINVAL, "null pointer argument");
  if (!c->has_bvh) return fail(SPLATS_ENOBVH, "splats_export_child_boxes before any update");
  if (!c->set[c->cur_set].has_exact)
    return fail(SPLATS_ESTATE, "splats_export_child_boxes: the exact node boxes were not stored by the last build (set SPLATS_OPT_EXACT_NODES before the update)");
  unsigned n = 0;
  int rc = splats_count(&n);
  if (rc) return rc;
  if (n < 2) return SPLATS_OK;
  // the first 48 bytes of every 64-byte record, exactly as the traversal reads them
  CU(cudaMemcpy2DAsync(child_boxes, 12 * sizeof(float), c->set[c->cur_set].nodes, sizeof(Node), 12 * sizeof(float), n - 1,
                       cudaMemcpyDeviceToDevice, c->stream));
  CU(cudaStreamSynchronize(c->stream));
  return SPLATS_OK;
}

int splats_export_qnodes(unsigned* qnodes, float* frame) {
  if (!g_ctx) return fail(SPLATS_ESTATE, "no context");
  Context* c = g_ctx;
  if (!c->has_bvh) return fail(SPLATS_ENOBVH, "splats_export_qnodes before any update");
  unsigned n = 0;
  int rc = splats_count(&n);
  if (rc) return rc;
  // the records exactly as the traversal reads them
  if (qnodes && n > 1) CU(cudaMemcpyAsync(qnodes, c->set[c->cur_set].qnodes, (size_t)(n - 1) * sizeof(QNode), cudaMemcpyDeviceToDevice, c->stream));
  if (frame) {   // bounds of the centres and the largest radius: what the quantisation frame is derived from
    FrameState hs;
    CU(cudaMemcpyAsync(&hs, c->state + c->cur_state, offsetof(FrameState, hist), cudaMemcpyDeviceToHost, c->stream));
    CU(cudaStreamSynchronize(c->stream));
    auto dec = [](uint32_t u) { uint32_t b = (u & 0x80000000u) ? (u & 0x7fffffffu) : ~u; float f; memcpy(&f, &b, 4); return f; };
    float h[7] = {0, 0, 0, 0, 0, 0, 0};
    if (n) {
      for (int a = 0; a < 3; ++a) { h[a] = dec(hs.lo[a]); h[3 + a] = dec(hs.hi[a]); }
      h[6] = dec(hs.rmax);
    }
    CU(cudaMemcpyAsync(frame, h, sizeof(h), cudaMemcpyHostToDevice, c->stream));
  }
  CU(cudaStreamSynchronize(c->stream));
  return SPLATS_OK;
}

int splats_export_splats(float* sphere, float* rgba, float* lo_hi) {
  if (!g_ctx) return fail(SPLATS_ESTATE, "no context");
  Context* c = g_ctx;
  if (!c->has_bvh) return fail(SPLATS_ENOBVH, "splats_export_splats before any update");
  unsigned n = 0;
  int rc = splats_count(&n);
  if (rc) return rc;
  if (sphere && n) CU(cudaMemcpyAsync(sphere, c->set[c->cur_set].sphere, (size_t)n * sizeof(float4), cudaMemcpyDeviceToDevice, c->stream));
  if (rgba && n) CU(cudaMemcpyAsync(rgba, c->set[c->cur_set].rgba, (size_t)n * sizeof(float4), cudaMemcpyDeviceToDevice, c->stream));
  if (lo_hi) {
    FrameState hs;
    CU(cudaMemcpyAsync(&hs, c->state + c->cur_state, sizeof(uint32_t) * 8, cudaMemcpyDeviceToHost, c->stream));
    CU(cudaStreamSynchronize(c->stream));
    float h[6];
    for (int a = 0; a < 3; ++a) {
      uint32_t ulo = hs.lo[a], uhi = hs.hi[a];
      uint32_t blo = (ulo & 0x80000000u) ? (ulo & 0x7fffffffu) : ~ulo;
      uint32_t bhi = (uhi & 0x80000000u) ? (uhi & 0x7fffffffu) : ~uhi;
      memcpy(&h[a], &blo, 4);
      memcpy(&h[3 + a], &bhi, 4);
      if (n == 0) h[a] = h[3 + a] = 0.0f;
    }
    CU(cudaMemcpyAsync(lo_hi, h, sizeof(h), cudaMemcpyHostToDevice, c->stream));
  }
  CU(cudaStreamSynchronize(c->stream));
  return SPLATS_OK;
}

int splats_set_option(int option, int value) {
  if (!g_ctx) return fail(SPLATS_ESTATE, "no context");
  switch (option) {
    case SPLATS_OPT_REFIT:
      if (value != SPLATS_REFIT_PYRAMID && value != SPLATS_REFIT_ATOMIC && value != SPLATS_REFIT_TILED) return fail(SPLATS_EINVAL, "unknown refit mode");
      g_ctx->refit_mode = value;
      return SPLATS_OK;
    case SPLATS_OPT_SORT:
      if (value != SPLATS_SORT_HYBRID && value != SPLATS_SORT_LSD8 && value != SPLATS_SORT_LSD8_LAUNCHES && value != SPLATS_SORT_HYBRID_LSD)
        return fail(SPLATS_EINVAL, "unknown sort mode");
      g_ctx->sort_mode = value;
      return SPLATS_OK;
    case SPLATS_OPT_OVERLAP:
      if (value != 0 && value != 1) return fail(SPLATS_EINVAL, "SPLATS_OPT_OVERLAP takes 0 or 1");
      g_ctx->overlap = value != 0;
      g_ctx->serialize_next_render = true;
      return SPLATS_OK;
    case SPLATS_OPT_EXACT_NODES:
      if (value != 0 && value != 1) return fail(SPLATS_EINVAL, "SPLATS_OPT_EXACT_NODES takes 0 or 1");
      g_ctx->exact_nodes = value != 0;
      return SPLATS_OK;
    case SPLATS_OPT_PDL:
      if (value != 0 && value != 1) return fail(SPLATS_EINVAL, "SPLATS_OPT_PDL takes 0 or 1");
      g_ctx->pdl = value != 0;
      return SPLATS_OK;
    default:
      return fail(SPLATS_EINVAL, "unknown option");
  }
}

int splats_set_radius(int mode, float param) {
  if (!g_ctx) return fail(SPLATS_ESTATE, "no context");
  if (mode != SPLATS_RADIUS_FOOTPRINT && mode != SPLATS_RADIUS_CONSTANT && mode != SPLATS_RADIUS_OPACITY)
    return fail(SPLATS_EINVAL, "unknown radius mode");
  if (mode == SPLATS_RADIUS_CONSTANT && !(param > 0.0f && std::isfinite(param)))
    return fail(SPLATS_EINVAL, "constant radius must be finite and > 0");
  if (mode == SPLATS_RADIUS_OPACITY && !(param >= 0.0f && param <= 1.0f))
    return fail(SPLATS_EINVAL, "opacity radius floor must be in [0, 1]");
  g_ctx->radius_mode = mode;
  g_ctx->radius_param = mode == SPLATS_RADIUS_FOOTPRINT ? 0.0f : param;
  return SPLATS_OK;
}

int splats_set_profiling(int on) {
  if (!g_ctx) return fail(SPLATS_ESTATE, "no context");
  g_ctx->profiling = on != 0;
  g_ctx->spans.clear();
  g_ctx->pool_used = 0;
  return SPLATS_OK;
}

int splats_stage_ms(float* ms_sum, unsigned* calls) {
  if (!g_ctx) return fail(SPLATS_ESTATE, "no context");
  if (!ms_sum) return fail(SPLATS_EINVAL, "null pointer argument");
  Context* c = g_ctx;
  CU(cudaStreamSynchronize(c->stream));
  for (int i = 0; i < SPLATS_NUM_STAGES; ++i) { ms_sum[i] = 0.0f; if (calls) calls[i] = 0; }
  for (const auto& sp : c->spans) {
    float ms = 0.0f;
    CU(cudaEventElapsedTime(&ms, c->pool[sp.e0], c->pool[sp.e1]));
    ms_sum[sp.stage] += ms;
    if (calls) calls[sp.stage] += 1;
  }
  c->spans.clear();
  c->pool_used = 0;
  return SPLATS_OK;
}

int splats_traced_pixels(unsigned long long* pixels_host, int reset) {
  if (!g_ctx) return fail(SPLATS_ESTATE, "no context");
  if (!pixels_host) return fail(SPLATS_EINVAL, "null pointer argument");
  Context* c = g_ctx;
  CU(cudaMemcpyAsync(pixels_host, c->traced, sizeof(unsigned long long), cudaMemcpyDeviceToHost, c->stream));
  if (reset) CU(cudaMemsetAsync(c->traced, 0, sizeof(unsigned long long), c->stream));
  CU(cudaStreamSynchronize(c->stream));
  return SPLATS_OK;
}

unsigned long long splats_launch_count(void) { return g_ctx ? g_ctx->launches : 0ull; }

int splats_synchronize(void) {
  if (!g_ctx) return fail(SPLATS_ESTATE, "no context");
  CU(cudaStreamSynchronize(g_ctx->stream));
  if (g_ctx->build_stream) CU(cudaStreamSynchronize(g_ctx->build_stream));
  if (g_ctx->h2d_stream) {
    CU(cudaStreamSynchronize(g_ctx->h2d_stream));
    CU(cudaStreamSynchronize(g_ctx->d2h_stream));
  }
  return SPLATS_OK;
}

#ifdef SPLATS_STATS
int splats_debug_stats(unsigned long long* out8, int reset) {
  if (!g_ctx) return fail(SPLATS_ESTATE, "no context");
  CU(cudaStreamSynchronize(g_ctx->stream));
  CU(cudaMemcpyFromSymbol(out8, sw::g_stats, sizeof(unsigned long long) * 8));
  if (reset) {
    unsigned long long z[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    CU(cudaMemcpyToSymbol(sw::g_stats, z, sizeof(z)));
  }
  return SPLATS_OK;
}
#endif

const char* splats_last_error(void) { return g_err.c_str(); }

void splats_destroy(void) {
  if (!g_ctx) return;
  cudaStreamSynchronize(g_ctx->stream);
  if (g_ctx->build_stream) cudaStreamSynchronize(g_ctx->build_stream);
  if (g_ctx->h2d_stream) { cudaStreamSynchronize(g_ctx->h2d_stream); cudaStreamSynchronize(g_ctx->d2h_stream); }
  free_all(g_ctx);
  delete g_ctx;
  g_ctx = nullptr;
}

}  // extern "C"
