// common.cuh -- shared device types and helpers of the splat-warp kernels (sm_100a).
//
// Arithmetic contract: every float32 operation that decides an integer
// (Morton code), a hit or a composited value is written with the explicit round-to-nearest
// intrinsics below, so nvcc can neither contract a*b+c into an FMA nor split an FMA that the
// spec asks for.  Slab tests are free (only conservative) and use ordinary operators.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace sw {

// ---- explicit IEEE float32 ops
__device__ __forceinline__ float fma_(float a, float b, float c) { return __fmaf_rn(a, b, c); }
__device__ __forceinline__ float mul_(float a, float b) { return __fmul_rn(a, b); }
__device__ __forceinline__ float add_(float a, float b) { return __fadd_rn(a, b); }
__device__ __forceinline__ float sub_(float a, float b) { return __fsub_rn(a, b); }
__device__ __forceinline__ float div_(float a, float b) { return __fdiv_rn(a, b); }
__device__ __forceinline__ float sqrt_(float a) { return __fsqrt_rn(a); }

// ---- programmatic dependent launch (sm_90+): a kernel launched with the stream-serialisation
// attribute may be scheduled while its predecessor in the stream is still draining; pdl_wait()
// blocks until that predecessor has completed and its writes are visible, so it must come
// before the first access to anything the predecessor produced.  Without the attribute both
// are no-ops.  pdl_trigger() lets the successor's blocks be scheduled once every block of this
// grid has started (they then sit in pdl_wait), which hides the launch latency between the
// short dependent kernels of one update.
// Which kernels release their dependent launch early (griddepcontrol.launch_dependents at their start) and which
// only when their blocks exit: 0 = all early; 1 = sort and tile kernel late; 2 = unproject too (default); 3 = spine
// too.  A dependent's blocks become resident as soon as they are released and spin in their wait: behind a short
// kernel that is harmless, behind a long one (sort, tile kernel) the waiting blocks take SM resources from the
// kernel they wait for.  Released at exit, the dependent's launch latency still hides behind the predecessor's tail.
#ifndef SPLATS_LATE_TRIGGER
#define SPLATS_LATE_TRIGGER 2
#endif
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_trigger() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

// ---- camera as kernel parameter (host fills the derived constants in float32)
struct DevCamera {
  float e[3], R[3], U[3], F[3];
  float tau;    // tan(fovy/2)
  float ta;     // fl(fl(tau*W)/H): horizontal half extent
  float fW, fH; // (float)W, (float)H
  int W, H;
};

// Ray through the centre of pixel (x, y), row 0 = top (Eq. 1's d):
// d = F + u R + v U, returned normalised together with the un-normalised length.
__device__ __forceinline__ void pixel_ray(const DevCamera& c, int x, int y, float d[3], float& len) {
  float nx = div_(__int2float_rn(2 * x + 1 - c.W), c.fW);
  float ny = div_(__int2float_rn(c.H - 2 * y - 1), c.fH);
  float u = mul_(nx, c.ta);
  float v = mul_(ny, c.tau);
#pragma unroll
  for (int k = 0; k < 3; ++k) d[k] = fma_(v, c.U[k], fma_(u, c.R[k], c.F[k]));
  len = sqrt_(fma_(d[2], d[2], fma_(d[1], d[1], mul_(d[0], d[0]))));
#pragma unroll
  for (int k = 0; k < 3; ++k) d[k] = div_(d[k], len);
}

__device__ __forceinline__ bool depth_valid(float t) {  // zero-radius samples are dropped
  return (t > 0.0f) && (t < __int_as_float(0x7f800000));
}

// Eq. 1: p = o + d t.
__device__ __forceinline__ void splat_centre(const DevCamera& c, int x, int y, float t, float p[3], float& len) {
  float d[3];
  pixel_ray(c, x, y, d, len);
#pragma unroll
  for (int k = 0; k < 3; ++k) p[k] = fma_(t, d[k], c.e[k]);
}

// ---- splat radius (S2 and its variants)
//   mode 0  footprint: r = k_r * z, k_r = (r_scale sqrt(1/2)) (2 tau / H)   (north_star)
//   mode 1  constant:  r = r_const = r_scale * param; the paper's choice, param = half a
//           voxel's diagonal
//   mode 2  opacity:   r = (k_r * z) * fma(w1, alpha, f_min), f_min = param, w1 = 1 - f_min
//           (a reading of PAPER.md:109 "varying the radius ... according to their opacity")
// All constants are computed on the host in float32, one rounding per operation.
struct RadiusParams {
  int mode;
  float k_r, r_const, f_min, w1;
};
__device__ __forceinline__ float splat_radius(const RadiusParams& rp, float z, float alpha) {
  if (rp.mode == 1) return rp.r_const;
  float r = mul_(rp.k_r, z);
  if (rp.mode == 2) r = mul_(r, fma_(rp.w1, alpha, rp.f_min));
  return r;
}

// ---- wire format (include/splats.h, wr_quant): 64-bit sample =
// x | y << 16 | z << 32 | radius << 48, four 16-bit fixed-point fields; colour = RGBA8.
struct QuantParams {
  float lo[3], ext[3];   // quantisation box and its extent hi - lo
  float cell[3];         // ext / 65536
  float r_max, rstep;    // radius of code 65535, r_max / 65535
};
__device__ __forceinline__ uint32_t quant_pos(float p, float lo, float ext) {
  const float s = mul_(div_(sub_(p, lo), ext), 65536.0f);
  if (!(s > 0.0f)) return 0u;
  if (s >= 65535.0f) return 65535u;
  return __float2uint_rz(s);
}
__device__ __forceinline__ uint32_t quant_radius(float r, float r_max) {  // rounded up, never 0
  const float u = ceilf(mul_(div_(r, r_max), 65535.0f));
  if (!(u > 1.0f)) return 1u;
  if (u >= 65535.0f) return 65535u;
  return __float2uint_rz(u);
}
__device__ __forceinline__ uint32_t quant_colour(float c) {
  const float x = fminf(fmaxf(c, 0.0f), 1.0f);
  return __float2uint_rz(add_(mul_(x, 255.0f), 0.5f));
}
__device__ __forceinline__ uint64_t pack_sample(const float p[3], float r, const QuantParams& q) {
  return (uint64_t)quant_pos(p[0], q.lo[0], q.ext[0]) | ((uint64_t)quant_pos(p[1], q.lo[1], q.ext[1]) << 16) |
         ((uint64_t)quant_pos(p[2], q.lo[2], q.ext[2]) << 32) | ((uint64_t)quant_radius(r, q.r_max) << 48);
}
__device__ __forceinline__ uint32_t pack_colour(const float4 c) {
  return quant_colour(c.x) | (quant_colour(c.y) << 8) | (quant_colour(c.z) << 16) | (quant_colour(c.w) << 24);
}
// centre of the sample's cell (a radius field of 0 marks a sample that must be dropped)
__device__ __forceinline__ void decode_centre(uint64_t w, const QuantParams& q, float p[3]) {
#pragma unroll
  for (int k = 0; k < 3; ++k)
    p[k] = fma_(add_(__uint2float_rn((uint32_t)(w >> (16 * k)) & 0xffffu), 0.5f), q.cell[k], q.lo[k]);
}
__device__ __forceinline__ float decode_radius(uint64_t w, const QuantParams& q) {
  return mul_(__uint2float_rn((uint32_t)(w >> 48)), q.rstep);
}
__device__ __forceinline__ float4 decode_colour(uint32_t c) {
  return make_float4(div_(__uint2float_rn(c & 0xffu), 255.0f), div_(__uint2float_rn((c >> 8) & 0xffu), 255.0f),
                     div_(__uint2float_rn((c >> 16) & 0xffu), 255.0f), div_(__uint2float_rn(c >> 24), 255.0f));
}

// ---- order-preserving float <-> uint32 map for atomicMin / atomicMax
__device__ __forceinline__ uint32_t f2ord(float f) {
  uint32_t u = __float_as_uint(f);
  return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}
__device__ __forceinline__ float ord2f(uint32_t u) {
  return __uint_as_float((u & 0x80000000u) ? (u & 0x7fffffffu) : ~u);
}

// ---- per-frame device state, double buffered by frame parity so that frame f can reset
// the accumulators of frame f+1 without a race or an extra launch.
struct FrameState {
  uint32_t lo[3];      // ordered-uint min of valid centres   (init 0xffffffff)
  uint32_t hi[3];      // ordered-uint max                     (init 0)
  uint32_t n;          // number of valid splats               (init 0)
  uint32_t pyr_done;   // blocks of leaf_pyramid_kernel that have finished (init 0)
  float root_lo[3];    // AABB of the whole scene (root node box), written by refit
  float root_hi[3];
  uint32_t sort_bar;       // grid barrier counter of the sort launch (init 0)
  uint32_t sort_fallback;  // set when the hybrid sort has to redo all 8 passes (init 0)
  uint32_t spine_n;        // nodes queued by tree_tile_kernel for tree_spine_kernel (init 0)
  uint32_t rmax;           // ordered-uint max of the valid splats' radii (init 0): with lo / hi the frame of the quantised node boxes
  uint32_t tile_done;      // blocks of tree_tile_kernel that have taken their pyramid ticket (init 0)
  uint32_t sort_wfall;     // set when a window of the windowed hybrid sort does not fit: fall back to the LSD passes (init 0)
  float qf[12];            // QFrame (lo, s, c; below) derived once per frame by unproject_kernel from lo / hi / rmax
  uint32_t hist[8][256];  // digit histograms of the 8 radix passes (init 0)
};

// ---- sort modes (onesweep.cuh) and what the producer of the keys must know about them
constexpr int SORT_HYBRID = 0, SORT_LSD8 = 1, SORT_SINGLE = 2, SORT_HYBRID_LSD = 3;
__host__ __device__ __forceinline__ bool sort_is_hybrid(int mode) { return mode == SORT_HYBRID || mode == SORT_HYBRID_LSD; }
// Which buffer unproject_kernel writes the unsorted pairs to, so that the sorted result always
// ends in buffer 0: the hybrid mode runs 4 passes (digits 4..7) up to HYBRID5_MIN elements and 5
// passes (digits 3..7) above it, where the cells of the top 31 bits are coarser than the sample
// pitch of a dense frame; an odd number of passes starts in buffer 1.
#ifndef SPLATS_HYBRID5_LOG
#define SPLATS_HYBRID5_LOG 19
#endif
constexpr uint32_t HYBRID5_MIN = 1u << SPLATS_HYBRID5_LOG;
__host__ __device__ __forceinline__ int hybrid_first_digit(uint32_t n) { return n > HYBRID5_MIN ? 3 : 4; }
// global passes of the windowed hybrid sort: the top 24 key bits, 32 above 2^23 splats (buckets stay at a few dozen keys)
__host__ __device__ __forceinline__ int win_passes(uint32_t n) { return n > (1u << 23) ? 4 : 3; }
__host__ __device__ __forceinline__ int sort_input_buffer(int mode, uint32_t n) {
  if (mode == SORT_HYBRID) return win_passes(n) & 1;   // the global passes end in buffer 0, where the buckets are put in order in place
  return (mode == SORT_HYBRID_LSD && (hybrid_first_digit(n) & 1)) ? 1 : 0;
}

// 64-byte BVH node: both child boxes live in the parent, so one node fetch (four 16-byte
// vector loads from one 64-byte-aligned record) tests both children.
//   b[0..5]  left child box  lo xyz, hi xyz      b[6..11] right child box
//   left/right: traversal links.  >= 0: internal node index (Karras numbering).  < 0: a
//     *leaf range*: the child subtree covers <= LEAF_MAX consecutive splats of the sorted
//     order, first | (count - 1) << 26 | 1 << 31; the traversal tests those spheres directly
//     instead of walking the subtree (a sphere test is far cheaper than a node visit).  The
//     canonical Karras links are recovered from the code: a range of 1 is the leaf `first`,
//     a longer left (right) range is internal node first + count - 1 (first).
//   parent: (parent index << 1) | is_right_child, -1 for the root
//   flag: arrival counter of the bottom-up refit
#ifndef SPLATS_LEAF_MAX
#define SPLATS_LEAF_MAX 1
#endif
constexpr int LEAF_MAX = SPLATS_LEAF_MAX;    // <= 32 (5-bit count field)
constexpr uint32_t LEAF_FIRST_MASK = (1u << 26) - 1;  // capacity: 2^26 - 1 splats
__host__ __device__ __forceinline__ uint32_t leaf_range_code(uint32_t first, uint32_t count) {
  return 0x80000000u | ((count - 1u) << 26) | first;
}
__host__ __device__ __forceinline__ uint32_t leaf_range_first(uint32_t code) { return code & LEAF_FIRST_MASK; }
__host__ __device__ __forceinline__ uint32_t leaf_range_count(uint32_t code) { return ((code >> 26) & 31u) + 1u; }

struct __align__(64) Node {
  float b[12];
  int left, right;
  int parent;
  unsigned flag;
};
static_assert(sizeof(Node) == 64, "node record must be 64 bytes");

// ---- traversal record (S13): 32 bytes, ONE 256-bit load per node visit.
// The twelve planes of the two child boxes are quantised to 16 bits over the frame
// [lo - rmax, hi + rmax] (lo / hi = bounds of the splat centres, rmax = largest radius: all three
// are known before the tree is built), lower planes rounded down, upper planes rounded up, so a
// quantised box always contains the exact one; the exact boxes are what the build computes
// (S7) and, with SPLATS_OPT_EXACT_NODES, also stores (Node).
//   w[a]     = q_lo | q_hi << 16 of axis a of the left child, w[3 + a] of the right child
//   w[6], w[7] = left / right link, as in Node
struct __align__(32) QNode {
  uint32_t w[8];
};
static_assert(sizeof(QNode) == 32, "traversal record must be 32 bytes");

struct QFrame {
  float lo[3];   // lo_a - rmax
  float s[3];    // 65535 / ext_a (encode), 0 for a zero extent
  float c[3];    // ext_a / 65535 (decode)
};
// derived once per frame (unproject_kernel, when lo / hi / rmax are final) and stored in FrameState::qf
__device__ __forceinline__ QFrame derive_qframe(const FrameState* st) {
  QFrame q;
  const float rmax = ord2f(st->rmax);
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    q.lo[a] = sub_(ord2f(st->lo[a]), rmax);
    const float ext = sub_(add_(ord2f(st->hi[a]), rmax), q.lo[a]);
    q.s[a] = ext > 0.0f ? div_(65535.0f, ext) : 0.0f;
    q.c[a] = div_(ext, 65535.0f);
  }
  return q;
}
__device__ __forceinline__ QFrame load_qframe(const FrameState* st) {
  QFrame q;
#pragma unroll
  for (int a = 0; a < 3; ++a) { q.lo[a] = __ldcg(&st->qf[a]); q.s[a] = __ldcg(&st->qf[3 + a]); q.c[a] = __ldcg(&st->qf[6 + a]); }
  return q;
}
// one axis of one child box: lower plane rounded down, upper plane rounded up, both clamped to 16 bits.
// floor / ceil without the conversion unit: for 0 <= u <= 65535, 2^23 + u rounded down (up) to float32 is
// 2^23 + floor(u) (ceil(u)) exactly, and its low mantissa bits are the integer.
__device__ __forceinline__ uint32_t quant_planes(float lo, float hi, float qlo, float s) {
  const float ul = fminf(fmaxf(mul_(sub_(lo, qlo), s), 0.0f), 65535.0f);   // fmaxf(NaN, 0) = 0
  const float uh = fminf(fmaxf(mul_(sub_(hi, qlo), s), 0.0f), 65535.0f);
  const uint32_t a = __float_as_uint(__fadd_rd(ul, 8388608.0f)), b = __float_as_uint(__fadd_ru(uh, 8388608.0f));
  return __byte_perm(a, b, 0x5410);   // a's low half | b's low half << 16
}
// L, R: lo xyz, hi xyz of the two child boxes
__device__ __forceinline__ void store_qnode(QNode* dst, const float* L, const float* R, int left, int right, const QFrame& q) {
  uint32_t w[8];
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    w[a] = quant_planes(L[a], L[3 + a], q.lo[a], q.s[a]);
    w[3 + a] = quant_planes(R[a], R[3 + a], q.lo[a], q.s[a]);
  }
  w[6] = (uint32_t)left;
  w[7] = (uint32_t)right;
  asm volatile("st.global.v8.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};"
               :: "l"(dst), "r"(w[0]), "r"(w[1]), "r"(w[2]), "r"(w[3]), "r"(w[4]), "r"(w[5]), "r"(w[6]), "r"(w[7]) : "memory");
}
// A box as six 16-bit codes in three words, arranged so that the union is three packed unsigned minima:
//   w0 = q_lo(x) | q_lo(y) << 16,  w1 = q_lo(z) | (65535 - q_hi(x)) << 16,  w2 = (65535 - q_hi(y)) | (65535 - q_hi(z)) << 16.
// Quantisation (floor for lower, ceil for upper planes of a monotone float32 expression) is monotone, so
// min / max commute with it: the tiled build carries boxes in this form from the leaves upwards and its
// records equal the quantised exact boxes bit for bit.
struct QBox {
  uint32_t w[3];
  __device__ __forceinline__ void init() { w[0] = w[1] = w[2] = 0xffffffffu; }
  __device__ __forceinline__ void merge(const QBox& o) {
#pragma unroll
    for (int i = 0; i < 3; ++i) w[i] = __vminu2(w[i], o.w[i]);
  }
  __device__ __forceinline__ QBox shfl_down(int delta) const {
    QBox o;
#pragma unroll
    for (int i = 0; i < 3; ++i) o.w[i] = __shfl_down_sync(0xffffffffu, w[i], delta);
    return o;
  }
  __device__ __forceinline__ QBox shfl_xor(int mask) const {
    QBox o;
#pragma unroll
    for (int i = 0; i < 3; ++i) o.w[i] = __shfl_xor_sync(0xffffffffu, w[i], mask);
    return o;
  }
};
__device__ __forceinline__ QBox quant_sphere(const float4 sp, const QFrame& q) {   // box of a splat: centre -+ radius (S2), quantised (S13)
  const uint32_t x = quant_planes(sub_(sp.x, sp.w), add_(sp.x, sp.w), q.lo[0], q.s[0]);
  const uint32_t y = quant_planes(sub_(sp.y, sp.w), add_(sp.y, sp.w), q.lo[1], q.s[1]);
  const uint32_t z = quant_planes(sub_(sp.z, sp.w), add_(sp.z, sp.w), q.lo[2], q.s[2]);
  QBox b;
  b.w[0] = __byte_perm(x, y, 0x5410);            // lo x | lo y << 16
  b.w[1] = __byte_perm(z, ~x, 0x7610);           // lo z | ~hi x << 16
  b.w[2] = __byte_perm(~y, ~z, 0x7632);          // ~hi y | ~hi z << 16
  return b;
}
// record words of one child: axis a -> q_lo | q_hi << 16
__device__ __forceinline__ void qbox_words(const QBox& b, uint32_t out[3]) {
  out[0] = __byte_perm(b.w[0], ~b.w[1], 0x7610);   // lo x | hi x << 16
  out[1] = __byte_perm(b.w[0], ~b.w[2], 0x5432);   // lo y | hi y << 16
  out[2] = __byte_perm(b.w[1], ~b.w[2], 0x7610);   // lo z | hi z << 16
}
__device__ __forceinline__ void store_qnode(QNode* dst, const QBox& L, const QBox& R, int left, int right) {
  uint32_t w[8];
  qbox_words(L, w);
  qbox_words(R, w + 3);
  w[6] = (uint32_t)left;
  w[7] = (uint32_t)right;
  asm volatile("st.global.v8.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};"
               :: "l"(dst), "r"(w[0]), "r"(w[1]), "r"(w[2]), "r"(w[3]), "r"(w[4]), "r"(w[5]), "r"(w[6]), "r"(w[7]) : "memory");
}
struct u8x { uint32_t v[8]; };
__device__ __forceinline__ u8x ldg_u8(const void* p) {   // read-only path (LDG.E.256.CONSTANT)
  u8x r;
  asm("ld.global.nc.v8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
      : "=r"(r.v[0]), "=r"(r.v[1]), "=r"(r.v[2]), "=r"(r.v[3]), "=r"(r.v[4]), "=r"(r.v[5]), "=r"(r.v[6]), "=r"(r.v[7]) : "l"(p));
  return r;
}

__device__ __forceinline__ uint64_t ld_volatile_u64(const uint64_t* p) {
  uint64_t v;
  asm volatile("ld.volatile.global.u64 %0, [%1];" : "=l"(v) : "l"(p));
  return v;
}
__device__ __forceinline__ void st_volatile_u64(uint64_t* p, uint64_t v) {
  asm volatile("st.volatile.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}

// 256-bit global accesses (sm_100): one request per 32 bytes instead of two, which halves the L1
// wavefronts of divergent 64-byte node fetches and scattered node writes.  32-byte aligned.
struct f8 { float v[8]; };
__device__ __forceinline__ f8 ldg_f8(const void* p) {   // read-only path (LDG.E.256.CONSTANT)
  f8 r;
  asm("ld.global.nc.v8.f32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
      : "=f"(r.v[0]), "=f"(r.v[1]), "=f"(r.v[2]), "=f"(r.v[3]), "=f"(r.v[4]), "=f"(r.v[5]), "=f"(r.v[6]), "=f"(r.v[7]) : "l"(p));
  return r;
}
__device__ __forceinline__ void stg_f8(void* p, const f8& r) {
  asm volatile("st.global.v8.f32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};"
               :: "l"(p), "f"(r.v[0]), "f"(r.v[1]), "f"(r.v[2]), "f"(r.v[3]), "f"(r.v[4]), "f"(r.v[5]), "f"(r.v[6]), "f"(r.v[7]) : "memory");
}

__device__ __forceinline__ float4 ldg_stream_f4(const float4* p) {  // read-once data: do not keep in L1
  float4 r;
  asm volatile("ld.global.nc.L1::no_allocate.v4.f32 {%0,%1,%2,%3}, [%4];"
               : "=f"(r.x), "=f"(r.y), "=f"(r.z), "=f"(r.w) : "l"(p));
  return r;
}

}  // namespace sw
