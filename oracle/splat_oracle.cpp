// oracle/splat_oracle.cpp -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// Plain, slow, single-threaded CPU statement of what the client hot path of
// arxiv 2006.14726 computes (2.5D frame -> sphere splats -> LBVH -> ray-traced,
// front-to-back composited image).  Only tests/, __graft_entry__.smoke() and
// bench.py's cpu_baseline / --impl reference legs may load it.  It shares no code
// with the CUDA path (paper_2006_14726_b200/csrc) and neither includes the other.
//
// Precision: float32 with the operation order written out below.  The paper does
// not fix a precision; the acceptance bar (BASELINE.json north_star) is *bit-exact*
// Morton codes / permutation / topology / AABBs, and a sphere hit-or-miss is a
// decision taken by floating point, so both sides take those decisions in the
// kernel's precision (float32) with one stated op order (DESIGN.md sec. 3,
// SURVEY.md sec. 8(c) O1..O9).  Compile with -ffp-contract=off: the only fused
// multiply-adds are the explicit fmaf() calls.
//
// Parity pins (tests/test_oracle_*.py): closed-form single-sphere hit t, closed-form
// alpha stack, identity-camera reprojection == source image bit-exactly, Morton codes
// vs a bit loop and hand-worked values, sort == numpy stable argsort, top-down tree
// == Karras' per-node construction (re-implemented in the test) on random and
// duplicate-heavy keys and on a hand-worked 8-key example, BVH-walk renderer ==
// brute-force renderer.  "Parity unpinned": only the conservative slab test used by
// the BVH-walk renderer (any conservative test is correct; it is checked through
// BVH-walk == brute force).
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <vector>

namespace {

struct Camera {  // PAPER.md:85 "the camera the buffers are associated with"
  float e[3], R[3], U[3], F[3], tau;
};

Camera load_camera(const float* c13) {
  Camera c;
  for (int k = 0; k < 3; ++k) { c.e[k] = c13[k]; c.R[k] = c13[3 + k]; c.U[k] = c13[6 + k]; c.F[k] = c13[9 + k]; }
  c.tau = c13[12];
  return c;
}

// O1 (first half) -- primary ray through the centre of pixel (x, y); row 0 = top.
// PAPER.md:63 sec. 4.1 "We march rays r = o + d t".  Returns the unit direction and
// the length `len` of the un-normalised direction F + u R + v U.
void pixel_ray(const Camera& c, int W, int H, int x, int y, float dhat[3], float* len_out) {
  float nx = (float)(2 * x + 1 - W) / (float)W;
  float ny = (float)(H - 2 * y - 1) / (float)H;
  float ta = (c.tau * (float)W) / (float)H;
  float u = nx * ta;
  float v = ny * c.tau;
  float d[3];
  for (int k = 0; k < 3; ++k) d[k] = fmaf(v, c.U[k], fmaf(u, c.R[k], c.F[k]));
  float len = sqrtf(fmaf(d[2], d[2], fmaf(d[1], d[1], d[0] * d[0])));
  for (int k = 0; k < 3; ++k) dhat[k] = d[k] / len;
  *len_out = len;
}

// O2 -- k_r = r_scale * sqrt(1/2) * (2 tau / H): half-diagonal of a pixel at unit
// view-axis depth (north_star: "radius is its one-pixel footprint at its depth";
// by analogy with PAPER.md:69 "half the size of a voxel's diagonal").
float radius_factor(const Camera& c, int H, float r_scale) {
  const float SQRT_HALF = 0.70710678118654752440f;
  return (r_scale * SQRT_HALF) * ((2.0f * c.tau) / (float)H);
}

// O2 variants.  mode 0: the footprint radius above.  mode 1: the
// paper's own choice, one radius for every sample -- "half the size of a voxel's diagonal"
// (PAPER.md:69); the caller passes that length as `param`, r = r_scale * param.  mode 2: a
// reading of the future-work idea "varying the radius of the object space samples according to
// their opacity": the footprint radius times f_min + (1 - f_min) * alpha, with
// f_min = param in [0, 1], so that opaque samples keep their footprint and faint ones shrink.
float splat_radius(int mode, float param, float r_scale, float k_r, float z, float alpha) {
  if (mode == 1) return r_scale * param;
  float r = k_r * z;
  if (mode == 2) {
    float w1 = 1.0f - param;
    r = r * fmaf(w1, alpha, param);
  }
  return r;
}

// O3 -- PAPER.md:69: samples with zero radius never reach the client.
bool depth_valid(float t) { return std::isfinite(t) && t > 0.0f; }

// O4 -- 63-bit Morton code, 21 bit per axis, x in the highest slot of each triple.
uint64_t morton63(const float c[3], const float lo[3], const float hi[3]) {
  uint32_t q[3];
  for (int k = 0; k < 3; ++k) {
    float ext = hi[k] - lo[k];
    if (ext > 0.0f) {
      float s = ((c[k] - lo[k]) / ext) * 2097152.0f;
      uint32_t v = (uint32_t)s;
      q[k] = v < 2097151u ? v : 2097151u;
    } else {
      q[k] = 0;
    }
  }
  uint64_t code = 0;
  for (int i = 0; i < 21; ++i) {
    code |= (uint64_t)((q[0] >> i) & 1u) << (3 * i + 2);
    code |= (uint64_t)((q[1] >> i) & 1u) << (3 * i + 1);
    code |= (uint64_t)((q[2] >> i) & 1u) << (3 * i);
  }
  return code;
}

// O8 -- ray / sphere entry point ("spheres that are represented as real quadrics",
// PAPER.md:55), perpendicular-vector form (the b*b - c form misses
// 9 % of the hits at these radii in float32).
bool ray_sphere(const float o[3], const float d[3], const float s[4], float* t_out) {
  float oc[3] = {s[0] - o[0], s[1] - o[1], s[2] - o[2]};
  float b = fmaf(oc[2], d[2], fmaf(oc[1], d[1], oc[0] * d[0]));
  float l[3];
  for (int k = 0; k < 3; ++k) l[k] = fmaf(-b, d[k], oc[k]);
  float l2 = fmaf(l[2], l[2], fmaf(l[1], l[1], l[0] * l[0]));
  float disc = fmaf(s[3], s[3], -l2);
  if (!(disc > 0.0f)) return false;  // tangent = miss
  float t = b - sqrtf(disc);
  if (!(t >= 0.0f)) return false;    // eye inside (or sphere behind): no contribution
  *t_out = t;
  return true;
}

struct Hit { float t; uint32_t id; uint32_t leaf; };
bool hit_less(const Hit& a, const Hit& b) { return a.t < b.t || (a.t == b.t && a.id < b.id); }

// O9 -- front-to-back premultiplied "over" of the hits in (t, id) order, stop once
// A >= 0.99 (tested after each hit).  "no shading other than the constant sample
// color".  Returns how many hits were composited.
int composite(std::vector<Hit>& hits, const float* rgba /*[N][4], sorted order*/, float out[4]) {
  std::sort(hits.begin(), hits.end(), hit_less);
  float C[3] = {0.0f, 0.0f, 0.0f}, A = 0.0f;
  int used = 0;
  for (const Hit& h : hits) {
    const float* col = rgba + 4 * (size_t)h.leaf;
    float T = 1.0f - A;
    for (int k = 0; k < 3; ++k) C[k] = fmaf(T, col[k], C[k]);
    A = fmaf(T, col[3], A);
    ++used;
    if (A >= 0.99f) break;
  }
  out[0] = C[0]; out[1] = C[1]; out[2] = C[2]; out[3] = A;
  return used;
}

// First-hit query -- the renderer the paper ships: "a simple first-hit ray tracing query and
// with no shading other than the constant sample color" (Fig. 2; sec. 4).
// The nearest accepted hit in (t, id) order supplies the pixel: its stored colour is copied,
// nothing is composited.  No hit: background (0,0,0,0).  Returns 1 if there was a hit.
int first_hit(const std::vector<Hit>& hits, const float* rgba /*[N][4], sorted order*/, float out[4]) {
  out[0] = out[1] = out[2] = out[3] = 0.0f;
  if (hits.empty()) return 0;
  const Hit* best = &hits[0];
  for (const Hit& h : hits)
    if (hit_less(h, *best)) best = &h;
  const float* col = rgba + 4 * (size_t)best->leaf;
  for (int k = 0; k < 4; ++k) out[k] = col[k];
  return 1;
}

// Conservative slab test for the BVH-walk renderer (unpinned on purpose): double
// arithmetic on a box padded by far more than the float32 error of ray_sphere().
bool ray_box_conservative(const float o[3], const float d[3], const float* box /*lo3,hi3*/) {
  double m = 1.0;
  for (int k = 0; k < 3; ++k) {
    m = std::max(m, std::fabs((double)o[k]));
    m = std::max(m, std::fabs((double)box[k]));
    m = std::max(m, std::fabs((double)box[3 + k]));
  }
  double pad = 1e-4 * m;
  double tn = -1e300, tf = 1e300;
  for (int k = 0; k < 3; ++k) {
    double lo = (double)box[k] - pad, hi = (double)box[3 + k] + pad;
    if (d[k] == 0.0f) {
      if (o[k] < lo || o[k] > hi) return false;
      continue;
    }
    double a = (lo - o[k]) / d[k], b = (hi - o[k]) / d[k];
    if (a > b) std::swap(a, b);
    tn = std::max(tn, a);
    tf = std::min(tf, b);
  }
  return tn <= tf && tf >= 0.0;
}

}  // namespace

extern "C" {

// ---- O1: unit ray direction of pixel (x, y) and the un-normalised length.
void oracle_pixel_ray(const float* cam13, int W, int H, int x, int y, float* dhat3, float* len) {
  Camera c = load_camera(cam13);
  pixel_ray(c, W, H, x, y, dhat3, len);
}

// ---- O1..O3: Eq. 1 p = o + d t_i for every pixel, radius, validity.
// sphere[p] = (cx, cy, cz, r) and valid[p]; entries of invalid pixels are zeroed.
// Returns N = number of valid pixels.
int64_t oracle_unproject(const float* depth, const float* cam13, int W, int H, float r_scale,
                         int radius_mode, float radius_param, const float* color /*[P][4], mode 2 only*/,
                         float* sphere /*[P][4]*/, uint8_t* valid /*[P]*/) {
  Camera c = load_camera(cam13);
  float k_r = radius_factor(c, H, r_scale);
  int64_t n = 0;
  for (int y = 0; y < H; ++y)
    for (int x = 0; x < W; ++x) {
      size_t p = (size_t)y * W + x;
      float t = depth[p];
      float* s = sphere + 4 * p;
      if (!depth_valid(t)) { valid[p] = 0; s[0] = s[1] = s[2] = s[3] = 0.0f; continue; }
      float dh[3], len;
      pixel_ray(c, W, H, x, y, dh, &len);
      for (int k = 0; k < 3; ++k) s[k] = fmaf(t, dh[k], c.e[k]);  // Eq. 1
      float z = t / len;                                          // view-axis depth
      s[3] = splat_radius(radius_mode, radius_param, r_scale, k_r, z, radius_mode == 2 ? color[4 * p + 3] : 0.0f);
      valid[p] = 1;
      ++n;
    }
  return n;
}

// ---- Wire format.  PAPER.md:69: "We quantize the object space
// coordinate and pack it together with the radius into 64 bits ... Before sending we compact
// that buffer by moving all the samples with zero radius to one side and send only those object
// space samples with non-zero radius"; "32 bits per color and 64 bits per object
// space sample (position and radius)".  The paper does not give the bit split; the reading taken
// (DESIGN.md sec. 2): four 16-bit fields, x | y << 16 | z << 32 | radius << 48; positions are
// fixed point over a quantisation box q = (lo[3], hi[3], r_max) that travels with the frame
// (cell = ext / 65536, decoded at the cell centre), the radius is fixed point over [0, r_max],
// rounded UP (a splat never shrinks) and never 0 for a kept sample; colour is RGBA8, rounded to
// nearest.  Compaction keeps ascending pixel order.
uint32_t quant_pos(float p, float lo, float ext) {
  float s = ((p - lo) / ext) * 65536.0f;
  if (!(s > 0.0f)) return 0u;
  if (s >= 65535.0f) return 65535u;
  return (uint32_t)s;
}
uint32_t quant_radius(float r, float r_max) {
  float u = ceilf((r / r_max) * 65535.0f);
  if (!(u > 1.0f)) return 1u;
  if (u >= 65535.0f) return 65535u;
  return (uint32_t)u;
}
uint32_t quant_colour(float c) {
  float x = fminf(fmaxf(c, 0.0f), 1.0f);
  return (uint32_t)(x * 255.0f + 0.5f);
}

// Server side: Eq. 1 + radius (as oracle_unproject) -> quantise -> pack -> compact.
// quant7 = lo xyz, hi xyz, r_max.  Returns the number of samples written.
int64_t oracle_pack(const float* color, const float* depth, const float* cam13, int W, int H, float r_scale,
                    int radius_mode, float radius_param, const float* quant7, uint64_t* samples /*[<=P]*/,
                    uint32_t* colours /*[<=P]*/) {
  size_t P = (size_t)W * H;
  std::vector<float> sphere(4 * P);
  std::vector<uint8_t> valid(P);
  oracle_unproject(depth, cam13, W, H, r_scale, radius_mode, radius_param, color, sphere.data(), valid.data());
  float ext[3];
  for (int k = 0; k < 3; ++k) ext[k] = quant7[3 + k] - quant7[k];
  int64_t n = 0;
  for (size_t p = 0; p < P; ++p) {
    const float* sp = sphere.data() + 4 * p;
    if (!valid[p] || !(sp[3] > 0.0f)) continue;   // zero radius: never sent
    uint64_t w = 0;
    for (int k = 0; k < 3; ++k) w |= (uint64_t)quant_pos(sp[k], quant7[k], ext[k]) << (16 * k);
    w |= (uint64_t)quant_radius(sp[3], quant7[6]) << 48;
    samples[n] = w;
    uint32_t c8 = 0;
    for (int k = 0; k < 4; ++k) c8 |= quant_colour(color[4 * p + k]) << (8 * k);
    colours[n] = c8;
    ++n;
  }
  return n;
}

// RGBA8 form of a float image (the display format of splats_render_rgba8): the wire's colour
// quantisation applied to every pixel.
void oracle_quantise_image(const float* rgba, int64_t n_pixels, uint32_t* out) {
  for (int64_t p = 0; p < n_pixels; ++p) {
    uint32_t c8 = 0;
    for (int k = 0; k < 4; ++k) c8 |= quant_colour(rgba[4 * p + k]) << (8 * k);
    out[p] = c8;
  }
}

// Client side: samples -> spheres (cx, cy, cz, r) and float colours, in the order received.
// A sample whose radius field is 0 is not a legal sample: valid[i] = 0 and it is dropped later.
void oracle_decode(const uint64_t* samples, const uint32_t* colours, int64_t n, const float* quant7,
                   float* sphere /*[n][4]*/, float* rgba /*[n][4]*/, uint8_t* valid /*[n]*/) {
  float cell[3];
  for (int k = 0; k < 3; ++k) cell[k] = (quant7[3 + k] - quant7[k]) / 65536.0f;
  float rstep = quant7[6] / 65535.0f;
  for (int64_t i = 0; i < n; ++i) {
    uint64_t w = samples[i];
    float* s = sphere + 4 * i;
    for (int k = 0; k < 3; ++k) {
      float q = (float)(uint32_t)((w >> (16 * k)) & 0xffffu);
      s[k] = fmaf(q + 0.5f, cell[k], quant7[k]);
    }
    uint32_t qr = (uint32_t)(w >> 48);
    s[3] = (float)qr * rstep;
    valid[i] = qr != 0u;
    if (!valid[i]) s[0] = s[1] = s[2] = s[3] = 0.0f;
    for (int k = 0; k < 4; ++k) rgba[4 * i + k] = (float)((colours[i] >> (8 * k)) & 0xffu) / 255.0f;
  }
}

// ---- O4 (bounds): component-wise min / max of the valid centres.
void oracle_bounds(const float* sphere, const uint8_t* valid, int64_t P, float* lo3, float* hi3) {
  bool any = false;
  for (int64_t p = 0; p < P; ++p) {
    if (!valid[p]) continue;
    const float* s = sphere + 4 * p;
    if (!any) { for (int k = 0; k < 3; ++k) lo3[k] = hi3[k] = s[k]; any = true; continue; }
    for (int k = 0; k < 3; ++k) { lo3[k] = fminf(lo3[k], s[k]); hi3[k] = fmaxf(hi3[k], s[k]); }
  }
  if (!any) for (int k = 0; k < 3; ++k) lo3[k] = hi3[k] = 0.0f;
}

uint64_t oracle_morton_point(const float* c3, const float* lo3, const float* hi3) { return morton63(c3, lo3, hi3); }

// ---- O3 + O4: compaction in ascending pixel order; ids[n] = pixel index, codes[n].
int64_t oracle_compact_codes(const float* sphere, const uint8_t* valid, int64_t P, const float* lo3,
                             const float* hi3, uint32_t* ids /*[N]*/, uint64_t* codes /*[N]*/) {
  int64_t n = 0;
  for (int64_t p = 0; p < P; ++p) {
    if (!valid[p]) continue;
    ids[n] = (uint32_t)p;
    codes[n] = morton63(sphere + 4 * p, lo3, hi3);
    ++n;
  }
  return n;
}

// ---- O5: std::stable_sort by code over ids in ascending order == order by (code, id).
// order[j] = compacted index of the j-th splat in sorted order.
void oracle_sort(const uint64_t* codes, int64_t N, uint32_t* order) {
  std::vector<uint32_t> idx((size_t)N);
  for (int64_t i = 0; i < N; ++i) idx[i] = (uint32_t)i;
  std::stable_sort(idx.begin(), idx.end(), [&](uint32_t a, uint32_t b) { return codes[a] < codes[b]; });
  for (int64_t i = 0; i < N; ++i) order[i] = idx[i];
}

// ---- O6: top-down binary radix tree over the sorted codes (LBVH, PAPER.md:71
// [LGS*09]), Karras numbering.  Node ids: internal j in [0, N-1) -> j, leaf i
// (sorted position) -> (N-1) + i.  children[j] = {left id, right id};
// parents[id] = internal index of the parent, -1 for the root;
// ranges[j] = {first, last} sorted position covered by internal node j.
void oracle_tree(const uint64_t* sorted_codes, int64_t N, int32_t* children /*[N-1][2]*/,
                 int32_t* parents /*[2N-1]*/, int32_t* ranges /*[N-1][2]*/) {
  if (N <= 0) return;
  if (N == 1) { parents[0] = -1; return; }  // the single leaf is the root
  struct Item { int64_t a, b; int32_t node; };
  std::vector<Item> stack;
  parents[0] = -1;
  stack.push_back({0, N - 1, 0});
  while (!stack.empty()) {
    Item it = stack.back();
    stack.pop_back();
    int64_t a = it.a, b = it.b, gamma = a;
    if (sorted_codes[a] != sorted_codes[b]) {
      uint64_t diff = sorted_codes[a] ^ sorted_codes[b];
      int m = 63;
      while (!((diff >> m) & 1ull)) --m;             // highest differing bit
      for (int64_t i = a; i <= b; ++i)               // last index whose bit m is 0
        if (!((sorted_codes[i] >> m) & 1ull)) gamma = i;
    } else {                                         // duplicates: split on the sorted position
      uint32_t diff = (uint32_t)a ^ (uint32_t)b;
      int m = 31;
      while (!((diff >> m) & 1u)) --m;
      for (int64_t i = a; i <= b; ++i)
        if (!(((uint32_t)i >> m) & 1u)) gamma = i;
    }
    int32_t left, right;
    if (gamma == a) left = (int32_t)(N - 1 + a);
    else { left = (int32_t)gamma; stack.push_back({a, gamma, left}); }
    if (gamma + 1 == b) right = (int32_t)(N - 1 + b);
    else { right = (int32_t)(gamma + 1); stack.push_back({gamma + 1, b, right}); }
    children[2 * (size_t)it.node] = left;
    children[2 * (size_t)it.node + 1] = right;
    parents[left] = it.node;
    parents[right] = it.node;
    ranges[2 * (size_t)it.node] = (int32_t)a;
    ranges[2 * (size_t)it.node + 1] = (int32_t)b;
  }
}

// ---- O7: leaf box = centre -/+ r; internal box = exact union of its children.
// sphere_sorted[i] = sphere of the leaf at sorted position i.  aabbs[id] = lo3, hi3.
void oracle_refit(const float* sphere_sorted, const int32_t* children, int64_t N, float* aabbs /*[2N-1][6]*/) {
  if (N <= 0) return;
  for (int64_t i = 0; i < N; ++i) {
    const float* s = sphere_sorted + 4 * i;
    float* bx = aabbs + 6 * (size_t)(N - 1 + i);
    for (int k = 0; k < 3; ++k) { bx[k] = s[k] - s[3]; bx[3 + k] = s[k] + s[3]; }
  }
  if (N == 1) return;
  // post-order over the tree (children before parents)
  std::vector<int32_t> order;
  std::vector<int32_t> stack{0};
  while (!stack.empty()) {
    int32_t j = stack.back();
    stack.pop_back();
    order.push_back(j);
    for (int s = 0; s < 2; ++s) {
      int32_t ch = children[2 * (size_t)j + s];
      if (ch < N - 1) stack.push_back(ch);
    }
  }
  for (size_t q = order.size(); q-- > 0;) {
    int32_t j = order[q];
    const float* l = aabbs + 6 * (size_t)children[2 * (size_t)j];
    const float* r = aabbs + 6 * (size_t)children[2 * (size_t)j + 1];
    float* bx = aabbs + 6 * (size_t)j;
    for (int k = 0; k < 3; ++k) { bx[k] = fminf(l[k], r[k]); bx[3 + k] = fmaxf(l[3 + k], r[3 + k]); }
  }
}

// ---- O8 for one ray and one sphere (pins: closed-form t).
int oracle_ray_sphere(const float* o3, const float* d3, const float* sphere4, float* t_out) {
  return ray_sphere(o3, d3, sphere4, t_out) ? 1 : 0;
}

// ---- O9 for a given hit list (pins: alpha-stack closed form).  rgba[i] belongs to hit i.
int oracle_composite(int n, const float* t, const uint32_t* id, const float* rgba, float* out4) {
  std::vector<Hit> hits((size_t)n);
  for (int i = 0; i < n; ++i) hits[i] = {t[i], id[i], (uint32_t)i};
  return composite(hits, rgba, out4);
}

// ---- L0: brute-force renderer -- every ray against every splat (the definition).
// Arrays are in sorted order (any order gives the same image: hits are ordered by
// (t, id)).  pixels == nullptr: whole frame into out[H2*W2*4]; otherwise only the
// n_pixels listed pixel indices, out[n_pixels*4].  hits_used (optional) receives the
// number of composited hits per output pixel.  first_hit_only != 0: the paper's first-hit
// query instead of compositing.
void oracle_render_brute(const float* sphere, const float* rgba, const uint32_t* ids, int64_t N,
                         const float* cam13, int W2, int H2, const int64_t* pixels, int64_t n_pixels,
                         int first_hit_only, float* out, int32_t* hits_used) {
  Camera c = load_camera(cam13);
  int64_t total = pixels ? n_pixels : (int64_t)W2 * H2;
  std::vector<Hit> hits;
  for (int64_t q = 0; q < total; ++q) {
    int64_t p = pixels ? pixels[q] : q;
    int x = (int)(p % W2), y = (int)(p / W2);
    float dh[3], len;
    pixel_ray(c, W2, H2, x, y, dh, &len);
    hits.clear();
    for (int64_t i = 0; i < N; ++i) {
      float t;
      if (ray_sphere(c.e, dh, sphere + 4 * i, &t)) hits.push_back({t, ids[i], (uint32_t)i});
    }
    int used = first_hit_only ? first_hit(hits, rgba, out + 4 * q) : composite(hits, rgba, out + 4 * q);
    if (hits_used) hits_used[q] = used;
  }
}

// ---- L1: the same image through a recursive walk of the oracle's own tree.
namespace {
void walk(int32_t id, int64_t N, const int32_t* children, const float* aabbs, const float* sphere,
          const uint32_t* ids, const float o[3], const float d[3], std::vector<Hit>& hits) {
  if (!ray_box_conservative(o, d, aabbs + 6 * (size_t)id)) return;
  if (id >= N - 1) {
    int64_t i = id - (N - 1);
    float t;
    if (ray_sphere(o, d, sphere + 4 * i, &t)) hits.push_back({t, ids[i], (uint32_t)i});
    return;
  }
  walk(children[2 * (size_t)id], N, children, aabbs, sphere, ids, o, d, hits);
  walk(children[2 * (size_t)id + 1], N, children, aabbs, sphere, ids, o, d, hits);
}
}  // namespace

void oracle_render_bvh(const float* sphere, const float* rgba, const uint32_t* ids, int64_t N,
                       const int32_t* children, const float* aabbs, const float* cam13, int W2, int H2,
                       const int64_t* pixels, int64_t n_pixels, int first_hit_only, float* out,
                       int32_t* hits_used) {
  Camera c = load_camera(cam13);
  int64_t total = pixels ? n_pixels : (int64_t)W2 * H2;
  std::vector<Hit> hits;
  for (int64_t q = 0; q < total; ++q) {
    int64_t p = pixels ? pixels[q] : q;
    int x = (int)(p % W2), y = (int)(p / W2);
    float dh[3], len;
    pixel_ray(c, W2, H2, x, y, dh, &len);
    hits.clear();
    if (N > 0) walk(0, N, children, aabbs, sphere, ids, c.e, dh, hits);
    int used = first_hit_only ? first_hit(hits, rgba, out + 4 * q) : composite(hits, rgba, out + 4 * q);
    if (hits_used) hits_used[q] = used;
  }
}

// ---- Server-side volume ray marcher (first half).  PAPER.md:63 sec. 4.1:
// "we render the volume using a ray marcher that employs one of the heuristics presented by
// Zellmann et al. to estimate which depth value represents the volume best.  We march rays
// r = o + d t"; it "writes out colors and t values to an off-screen buffer".  The
// paper gives neither its transfer function nor the heuristic's formula; the reading is
// BASELINE.json's server pass: unit cube, n^3 float32 densities at voxel
// centres, trilinear, clamp to edge, samples at t0 + (s + 1/2) * step with step = 0.5 / n,
// opacity tents, premultiplied front-to-back compositing, depth = t of the first sample at which
// the accumulated alpha reaches depth_alpha (0 if never: dropped), stop at stop_alpha.  float32
// with the operation order of DESIGN.md S12.  tf = n_tents, then iso[4], alpha[4], rgb[4][3],
// half_width, shade, depth_alpha, stop_alpha (all float32; layout of wr_transfer).
static inline float lerp1(float a, float b, float f) { return fmaf(f, b - a, a); }

void oracle_march(const float* vol, int n, const int32_t* tf_n, const float* tf, const float* cam13, int W, int H,
                  float* color /*[H*W*4]*/, float* depth /*[H*W]*/) {
  Camera c = load_camera(cam13);
  const int nt = *tf_n;
  const float* iso = tf; const float* amax = tf + 4; const float* rgb = tf + 8;
  const float hw = tf[20], shade = tf[21], depth_alpha = tf[22], stop_alpha = tf[23];
  const float one_minus_shade = 1.0f - shade;
  const float fn = (float)n, step = 0.5f / fn;
  for (int y = 0; y < H; ++y)
    for (int x = 0; x < W; ++x) {
      size_t p = (size_t)y * W + x;
      float d[3], len;
      pixel_ray(c, W, H, x, y, d, &len);
      float t0 = 0.0f, t1 = INFINITY;
      bool miss = false;
      for (int k = 0; k < 3; ++k) {
        if (fabsf(d[k]) < 1e-30f) {
          if (c.e[k] < 0.0f || c.e[k] > 1.0f) miss = true;
          continue;
        }
        float a = (0.0f - c.e[k]) / d[k], b = (1.0f - c.e[k]) / d[k];
        if (a > b) { float s = a; a = b; b = s; }
        t0 = fmaxf(t0, a);
        t1 = fminf(t1, b);
      }
      float C[3] = {0.0f, 0.0f, 0.0f}, A = 0.0f, tdepth = 0.0f;
      if (!miss && t0 < t1) {
        for (int s = 0;; ++s) {
          float t = fmaf((float)s + 0.5f, step, t0);
          if (!(t < t1)) break;
          float P[3], f[3];
          int i0[3], i1[3];
          for (int k = 0; k < 3; ++k) {
            P[k] = fmaf(t, d[k], c.e[k]);
            float g = fmaf(P[k], fn, -0.5f);
            float fl = floorf(g);
            f[k] = g - fl;
            int a = (int)fl, b = a + 1;
            a = a < 0 ? 0 : (a > n - 1 ? n - 1 : a);
            b = b < 0 ? 0 : (b > n - 1 ? n - 1 : b);
            i0[k] = a; i1[k] = b;
          }
          auto V = [&](int i, int j, int k) -> float { return vol[((size_t)k * n + j) * n + i]; };
          float c00 = lerp1(V(i0[0], i0[1], i0[2]), V(i1[0], i0[1], i0[2]), f[0]);
          float c10 = lerp1(V(i0[0], i1[1], i0[2]), V(i1[0], i1[1], i0[2]), f[0]);
          float c01 = lerp1(V(i0[0], i0[1], i1[2]), V(i1[0], i0[1], i1[2]), f[0]);
          float c11 = lerp1(V(i0[0], i1[1], i1[2]), V(i1[0], i1[1], i1[2]), f[0]);
          float dens = lerp1(lerp1(c00, c10, f[1]), lerp1(c01, c11, f[1]), f[2]);
          float alpha = 0.0f;
          int ci = -1;
          for (int i = 0; i < nt; ++i) {
            float w = 1.0f - fabsf(dens - iso[i]) / hw;
            if (w > 0.0f) {
              alpha = fmaf(amax[i], w, alpha);
              if (ci < 0) ci = i;
            }
          }
          if (alpha > 0.0f) {
            float T = 1.0f - A, Ta = T * alpha;
            for (int k = 0; k < 3; ++k) {
              float pc = fminf(fmaxf(P[k], 0.0f), 1.0f);
              float mod = fmaf(shade, pc, one_minus_shade);
              C[k] = fmaf(Ta, rgb[3 * ci + k] * mod, C[k]);
            }
            A = fmaf(T, alpha, A);
            if (tdepth == 0.0f && A >= depth_alpha) tdepth = t;
            if (A >= stop_alpha) break;
          }
        }
      }
      color[4 * p + 0] = C[0]; color[4 * p + 1] = C[1]; color[4 * p + 2] = C[2]; color[4 * p + 3] = A;
      depth[p] = tdepth;
    }
}

// ---- Comparison renderer: the 2.5D point rendering of [ZAL12] that
// the paper compares against -- "the authors render the image pixels as point primitives"
// (PAPER.md:37), object space coordinate -> "window coordinates by applying the viewing and
// camera transforms as well as viewport transform", "the point primitives' size is
// fixed to a certain number of pixels", depth test "not performed per fragment but
// per vertex".  Restated without a graphics API: every splat centre is projected
// with the destination camera; it covers the point_px x point_px pixels whose centres lie in the
// square (w - size/2, w + size/2] of that side around its window position (the OpenGL point
// rasterisation rule: odd sizes centre on floor(w) + 1/2, even sizes on floor(w + 1/2)); each
// pixel shows the stored colour of the covering point with the smallest view-axis depth (ties:
// smaller splat id); no blending; points at or behind the eye plane are culled.
void oracle_render_points(const float* sphere, const float* rgba, const uint32_t* ids, int64_t N,
                          const float* cam13, int W2, int H2, int point_px, float* out /*[H2*W2*4]*/) {
  Camera c = load_camera(cam13);
  size_t P2 = (size_t)W2 * H2;
  std::vector<float> zbuf(P2, 0.0f);
  std::vector<int64_t> owner(P2, -1);
  float ta = (c.tau * (float)W2) / (float)H2;
  float hW = 0.5f * (float)W2, hH = 0.5f * (float)H2;
  float off = 0.5f * (float)point_px + 0.5f;
  for (int64_t i = 0; i < N; ++i) {
    const float* s = sphere + 4 * i;
    float v[3] = {s[0] - c.e[0], s[1] - c.e[1], s[2] - c.e[2]};
    float zc = fmaf(v[2], c.F[2], fmaf(v[1], c.F[1], v[0] * c.F[0]));
    if (!(zc > 0.0f)) continue;
    float xr = fmaf(v[2], c.R[2], fmaf(v[1], c.R[1], v[0] * c.R[0]));
    float yu = fmaf(v[2], c.U[2], fmaf(v[1], c.U[1], v[0] * c.U[0]));
    float ndx = xr / (zc * ta), ndy = yu / (zc * c.tau);
    float wx = fmaf(ndx, hW, hW), wy = fmaf(-ndy, hH, hH);
    float fx0 = floorf(wx - off) + 1.0f, fy0 = floorf(wy - off) + 1.0f;
    if (!(fx0 > -1e9f && fx0 < 1e9f && fy0 > -1e9f && fy0 < 1e9f)) continue;   // far off screen / not finite
    long x0 = (long)fx0, y0 = (long)fy0;
    for (long y = y0; y < y0 + point_px; ++y)
      for (long x = x0; x < x0 + point_px; ++x) {
        if (x < 0 || y < 0 || x >= W2 || y >= H2) continue;
        size_t p = (size_t)y * W2 + x;
        bool wins = owner[p] < 0 || zc < zbuf[p] || (zc == zbuf[p] && ids[i] < ids[owner[p]]);
        if (wins) { zbuf[p] = zc; owner[p] = i; }
      }
  }
  for (size_t p = 0; p < P2; ++p)
    for (int k = 0; k < 4; ++k) out[4 * p + k] = owner[p] < 0 ? 0.0f : rgba[4 * (size_t)owner[p] + k];
}

}  // extern "C"
