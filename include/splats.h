/* splats.h -- C ABI of the B200-native client hot path of arxiv 2006.14726
 * (Zellmann, "Augmenting Image Warping-Based Remote Volume Rendering with Ray Tracing").
 *
 * The path (PAPER.md = the paper's text; SURVEY.md sec. 8 = the scope table):
 *   2.5D frame (RGBA + one depth per pixel, sec. 2; sec. 4.2)
 *   -> object-space sphere splats, Eq. 1 p = o + d t_i with a footprint
 *      radius
 *   -> LBVH over the spheres, rebuilt whenever a frame arrives
 *   -> software ray tracing of the spheres from the current camera (sec. 4),
 *      here with front-to-back compositing of every hit (BASELINE.json north_star).
 *
 * Conventions common to all calls
 *   - One library-wide context (created by splats_create, destroyed by splats_destroy); the
 *     calls are not thread-safe against each other.
 *   - "dev" pointers are CUDA device pointers on the device that was current at
 *     splats_create; "host" pointers are ordinary host memory (pinned memory makes the
 *     *_host copies asynchronous).  The caller owns every buffer it passes in; the library
 *     owns splats, keys, two BVH sets and scratch, all allocated once in splats_create (about
 *     275 bytes per capacity pixel; the staging of the *_host calls, 88 bytes per pixel, and the
 *     stream of splats_update_begin are created on first use).
 *   - splats_update / splats_render only ENQUEUE work on the stream given to splats_create and
 *     return; input/output buffers must stay valid until that work has run.  No allocation
 *     and no host<->device synchronisation happens on those two calls.
 *   - Return value: 0 = ok, SPLATS_EINVAL (-1) invalid argument, SPLATS_ENOBVH (-2) render
 *     before any update, SPLATS_ECUDA (-3) CUDA error, SPLATS_ESTATE (-4) no context /
 *     context already exists / call not allowed while a splats_update_begin is pending.
 *     splats_last_error() gives the text.  Nothing aborts or throws.
 *   - There is no CPU fallback: without a CUDA device splats_create fails with SPLATS_ECUDA.
 */
#ifndef SPLATS_H_
#define SPLATS_H_

#ifdef __cplusplus
extern "C" {
#endif

#define SPLATS_OK       0
#define SPLATS_EINVAL  (-1)
#define SPLATS_ENOBVH  (-2)
#define SPLATS_ECUDA   (-3)
#define SPLATS_ESTATE  (-4)

/* "the camera the buffers are associated with".  POD, host memory, 13 floats.
 * right/up/fwd must be an orthonormal basis of unit vectors; tan_half_fovy = tan(fovy/2) is
 * computed by the caller (device code uses no transcendentals).  The aspect ratio is W/H of
 * the call the camera is passed to.  Pixel (x, y), row 0 = top, has its centre at
 * ndc ((2x+1-W)/W, (H-2y-1)/H); its ray is fwd + ndc_x*tan*W/H*right + ndc_y*tan*up. */
typedef struct {
  float eye[3];
  float right[3];
  float up[3];
  float fwd[3];
  float tan_half_fovy;
} wr_camera;

/* Allocate all device memory for source frames of up to max_W*max_H pixels (< 2^26) and
 * destination images of up to the same pixel count.  cuda_stream: a cudaStream_t (NULL = the
 * legacy default stream) on which every later call enqueues its work. */
int splats_create(void* cuda_stream, int max_W, int max_H);

/* Frame received ("The client upon receiving the data will build an LBVH"):
 * unproject every valid pixel into a sphere splat and build the LBVH over all splats.
 *   color  dev, H*W*4 float32, premultiplied RGBA, row-major, row 0 = top; 16-byte aligned
 *   depth  dev, H*W float32: ray parameter t_i of Eq. 1 for a unit-length ray direction
 *          (distance from the eye); t <= 0, NaN or Inf marks a dropped pixel (PAPER.md:69:
 *          zero-radius samples are never sent); 16-byte aligned
 *   src_camera  host; the camera the frame was rendered from
 *   r_scale     > 0; splat radius = r_scale * half-diagonal of the pixel's footprint at the
 *               splat's view-axis depth (north_star)
 * Steps: bounds, unproject+Morton+compaction, onesweep radix
 * sort by (code, id), Karras hierarchy, bottom-up refit.  W*H = 0 valid pixels is not an
 * error (the next render writes zeros).
 * Errors: EINVAL for NULL pointers, W*H outside [1, capacity], non-finite or <= 0 r_scale,
 * non-finite camera. */
int splats_update(const float* color, const float* depth, const wr_camera* src_camera,
                  int W, int H, float r_scale);

/* Decoupled build.  The paper's client keeps displaying warped frames while the next server frame
 * is on its way ("decoupled the rendering and display phases"; requests are "handled
 * in threads separate from the main rendering thread").  splats_update_begin is
 * splats_update on a stream of the library: the build starts after everything enqueued so far
 * on the caller's stream, writes a second BVH, and does not hold up what the caller enqueues
 * next -- splats_render* keep reading the current BVH and may run at the same time.
 * splats_update_commit makes the new BVH the current one: everything enqueued afterwards waits
 * for the build.  Results are those of splats_update.  Between begin and commit: the input
 * buffers must stay valid and unchanged; splats_update*, a second begin and splats_export fail
 * with SPLATS_ESTATE.  Arguments and other errors as splats_update.  (Measured on B200: the build
 * does not get faster or slower this way and a step of the benchmark takes the same time, because
 * the persistent render blocks leave no room for the sort's 128-register blocks on an SM; what
 * the pair buys is that the renders of the current BVH are not delayed by an arriving frame.)
 * Progress: the sort of the build is a co-resident grid that spins on a grid barrier; beside a
 * persistent render grid it is scheduled as render blocks retire, so it advances because renders
 * END -- never enqueue a render that waits (on an event or a host callback) for a pending build. */
int splats_update_begin(const float* color, const float* depth, const wr_camera* src_camera,
                        int W, int H, float r_scale);
int splats_update_commit(void);

/* Display frame ("the current pixel buffer is warped according to the new
 * transformation"; ray trace the spheres): one primary ray per destination
 * pixel through the BVH of the latest splats_update, every sphere entry hit ordered by
 * (t, splat id) and composited front to back (premultiplied "over") until alpha >= 0.99.
 *   out_rgba  dev, H2*W2*4 float32, premultiplied, background (0,0,0,0); 16-byte aligned
 * W2 x H2 may differ from the source frame's size (W2*H2 <= capacity).
 * Errors: EINVAL as above, ENOBVH if no update was enqueued yet. */
int splats_render(const wr_camera* dst_camera, int W2, int H2, float* out_rgba);

/* The paper's own display query (sec. 4: "we render using first-hit ray tracing";
 * PAPER.md:59 Fig. 2: "a simple first-hit ray tracing query and with no shading other than the
 * constant sample color"): every destination pixel receives the
 * stored colour of the sphere whose entry point is nearest along its ray -- order (t, splat
 * id), same hit definition as splats_render -- and (0,0,0,0) if the ray enters no sphere.
 * Nothing is composited.  Arguments, layout and errors as splats_render. */
int splats_render_first_hit(const wr_camera* dst_camera, int W2, int H2, float* out_rgba);

/* The renderer the paper compares against ("we implemented the reference method by
 * Zellmann et al. using OpenGL point rendering"), restated as CUDA
 * kernels because no graphics API exists on this machine: the centres of the splats of the
 * latest update are projected with dst_camera to window coordinates and drawn as
 * square points of point_px x point_px pixels (a size "fixed to a certain number of
 * pixels"; OpenGL's rule: pixel centres in (w - size/2, w + size/2]), depth-tested per point
 * on the view-axis depth, ties to the smaller splat id, no blending: each pixel
 * shows the stored colour of its nearest point, background (0,0,0,0).  Points at or behind the
 * eye plane are culled.  point_px in [1, 64].  Arguments, layout, errors as splats_render. */
int splats_render_points(const wr_camera* dst_camera, int W2, int H2, int point_px, float* out_rgba);

/* ---- The paper's wire format -------------------------------------
 * the server sends "object space samples ... comprised of the coordinates from
 * Equation 1 and a footprint radius.  We quantize the object space coordinate and pack it
 * together with the radius into 64 bits", compacted so that only samples with non-zero radius
 * travel; "32 bits per color and 64 bits per object space sample".  The paper
 * does not print the bit split; this library's reading:
 *   sample  uint64 = qx | qy << 16 | qz << 32 | qr << 48, four unsigned 16-bit fields;
 *           q_k = clamp(floor((p_k - lo_k) / (hi_k - lo_k) * 65536), 0, 65535), decoded at the cell
 *           centre lo_k + (q_k + 0.5) * (hi_k - lo_k) / 65536;
 *           qr = clamp(ceil(r / r_max * 65535), 1, 65535), decoded as qr * (r_max / 65535): the
 *           radius is rounded up, and a field of 0 never occurs in a sample that is sent
 *   colour  uint32 = R | G << 8 | B << 16 | A << 24, round(255 * clamp(c, 0, 1)), decoded c / 255
 * wr_quant (host memory) is the frame header both sides must agree on: the quantisation box
 * (e.g. the volume's bounding box) and the largest representable radius. */
typedef struct {
  float lo[3];
  float hi[3];
  float r_max;
} wr_quant;

/* Server side, first half: the volume ray marcher (sec. 4.1 "we render the volume
 * using a ray marcher that employs one of the heuristics presented by Zellmann et al. to estimate
 * which depth value represents the volume best.  We march rays r = o + d t"; PAPER.md:85 it
 * "writes out colors and t values to an off-screen buffer").  The paper prints neither its
 * transfer function nor the heuristic; the reading is BASELINE.json's server pass:
 *   volume   dev, n*n*n float32 densities, x fastest, at the voxel centres of the unit cube
 *            [0,1]^3; sampled trilinearly, clamped to the edge, at t0 + (s + 1/2) * 0.5/n
 *   tf       host; opacity = sum over tents of alpha[i] * max(0, 1 - |density - iso[i]| /
 *            half_width); colour = rgb of the lowest tent with a positive weight, times
 *            (1 - shade + shade * clamp(position, 0, 1)) per channel; no opacity correction
 *   color    dev out, H*W*4 float32: premultiplied front-to-back composite, 16-byte aligned
 *   depth    dev out, H*W float32: ray parameter t (unit direction) of the first sample at which
 *            the accumulated alpha is >= depth_alpha, 0 if never (a dropped pixel); the march
 *            stops once the accumulated alpha is >= stop_alpha
 * The outputs are exactly what splats_update / splats_pack take.  Only enqueues.  Errors:
 * EINVAL (null pointers, n outside [1, 2048], n_tents outside [1, 4], half_width <= 0, W*H
 * outside [1, capacity], bad camera). */
typedef struct {
  int n_tents;
  float iso[4];
  float alpha[4];
  float rgb[4][3];
  float half_width;
  float shade;
  float depth_alpha;
  float stop_alpha;
} wr_transfer;
int splats_march(const float* volume, int n, const wr_transfer* tf, const wr_camera* camera, int W,
                 int H, float* color, float* depth);

/* Server side, second half: Eq. 1 + radius (mode of splats_set_radius) for every pixel of the 2.5D frame,
 * quantise, pack, and compact in ascending pixel order (the step the paper runs serially on
 * the CPU: 23 ms at 1024 x 1024).  Only enqueues.
 *   color, depth, src_camera, W, H, r_scale   as splats_update
 *   samples  dev, room for W*H uint64; colors  dev, room for W*H uint32; 16-byte aligned
 *   count    dev, one uint32: the number of samples written (pixels with a valid depth and a
 *            radius > 0)
 * Uses scratch of the context (W*H <= capacity).  Errors: EINVAL as splats_update, or for a
 * box with hi <= lo / non-finite values / r_max <= 0. */
int splats_pack(const float* color, const float* depth, const wr_camera* src_camera, int W, int H,
                float r_scale, const wr_quant* quant, unsigned long long* samples, unsigned* colors,
                unsigned* count);

/* splats_pack for callers that must not allocate: no context, no cudaMalloc / cudaFree / allocating
 * library call, usable without splats_create (code under CUDA graph capture, tight serving loops,
 * harnesses that forbid allocation).  Same result as splats_pack, bit for bit; the per-tile counts
 * of the compaction, which splats_pack keeps in scratch memory of the context, live in a
 * file-scope `static __device__` array of the library instead: 32 KiB, held by every GPU that
 * loads the library until the process exits.
 *   radius_mode, radius_param   as splats_set_radius (there is no context to read them from)
 *   cuda_stream                 cudaStream_t (NULL = the default stream) the two launches go to
 *   everything else             as splats_pack
 * Limit: W*H <= SPLATS_NOALLOC_MAX_PIXELS (4096 x 4096); beyond it the call fails with EINVAL and
 * does nothing.  The array is shared by every call and keeps the last call's contents; every
 * word a call reads it has written first, so nothing has to be cleared -- but two calls that
 * overlap on the GPU (different streams, or one device from two threads) race on it: serialise
 * them.  The array's device address is looked up once per device (cudaGetSymbolAddress, with that
 * device current) on the first call there, or ahead of time by splats_noalloc_setup (e.g. before
 * a capture begins).  Errors: EINVAL (null / misaligned pointers, sizes, camera, r_scale, radius
 * mode, box), ECUDA. */
#define SPLATS_NOALLOC_MAX_PIXELS (4096 * 4096)
int splats_noalloc_setup(void);
int splats_pack_noalloc(const float* color, const float* depth, const wr_camera* src_camera, int W, int H,
                        float r_scale, int radius_mode, float radius_param, const wr_quant* quant,
                        unsigned long long* samples, unsigned* colors, unsigned* count, void* cuda_stream);

/* Client side, the paper's literal entry point ("The client upon receiving the
 * data will build an LBVH"): build the splats and the BVH from n received samples.  Splat ids are
 * positions in the buffer; a sample whose radius field is 0 is dropped.  The buffers must stay
 * valid until the enqueued work has run.  n = 0 is allowed (the next render writes zeros).
 *   samples  dev, n uint64, 16-byte aligned;  colors  dev, n uint32;  n <= capacity
 * Afterwards splats_render / splats_render_first_hit / splats_export work as after
 * splats_update.  Errors: EINVAL (null pointers with n > 0, n > capacity, bad quant). */
int splats_update_packed(const unsigned long long* samples, const unsigned* colors, unsigned n,
                         const wr_quant* quant);

/* splats_update_packed with HOST buffers: what the paper's client does when a frame arrives from
 * the network -- 12 bytes per sample cross PCIe instead of 20 bytes per pixel.
 * Pipelined like splats_update_host (the buffers must stay valid until splats_synchronize). */
int splats_update_packed_host(const unsigned long long* samples_host, const unsigned* colors_host,
                              unsigned n, const wr_quant* quant);

/* The same two calls with HOST buffers (end-to-end path).  Both only ENQUEUE and return: the
 * frame is uploaded on a copy stream of the library into one of two device staging buffers,
 * the kernels wait for it on the compute stream, and each rendered image is read back on a
 * second copy stream from one of three device staging buffers, so the upload of the next
 * frame and the read-back of the previous image overlap the kernels.  Pinned host memory
 * makes the copies asynchronous.  The host buffers must stay valid, and out_rgba_host is
 * complete, only after splats_synchronize().  Results are bit-identical to the device calls. */
int splats_update_host(const float* color_host, const float* depth_host,
                       const wr_camera* src_camera, int W, int H, float r_scale);
int splats_render_host(const wr_camera* dst_camera, int W2, int H2, float* out_rgba_host);

/* splats_render with an 8-bit image: every pixel is written as one uint32 R | G << 8 | B << 16 |
 * A << 24 with round(255 * clamp(c, 0, 1)) per channel of the composited premultiplied colour
 * (the colour format of the wire, "32 bits per color") -- what a client that only
 * displays the warped frame needs, at a quarter of the bytes.  out_rgba8: dev (or host for the
 * _host variant, same pipelining as splats_render_host), H2*W2 uint32.  Errors as splats_render. */
int splats_render_rgba8(const wr_camera* dst_camera, int W2, int H2, unsigned* out_rgba8);
int splats_render_host_rgba8(const wr_camera* dst_camera, int W2, int H2, unsigned* out_rgba8_host);

/* Number of splats N of the latest update.  Synchronises the stream.  Parity/debug only. */
int splats_count(unsigned* n_host);

/* Export the BVH of the latest update in canonical form for the bit-exact acceptance
 * checks.  All pointers are dev pointers (any may be NULL to skip it); synchronises.
 *   keys        N  uint64   sorted 63-bit Morton codes
 *   perm        N  uint32   splat ids (= source pixel indices) in sorted order
 *   children    (N-1)*2 int32; node ids: internal j -> j, leaf at sorted position i -> N-1+i
 *   parents     (2N-1) int32, indexed by node id; -1 for the root
 *   node_aabbs  (2N-1)*6 float32: lo xyz, hi xyz per node id -- the EXACT boxes (oracle step O7).
 *               The traversal reads 16-bit quantised boxes (splats_export_qnodes) and the default
 *               (tiled) build forms nothing else; the exact boxes exist only while
 *               SPLATS_OPT_EXACT_NODES is on: without it node_aabbs != NULL fails with ESTATE.
 * Internal nodes use Karras' numbering (root 0; an internal child covering sorted range
 * [a,g] is node g when it is a left child, node a when it is a right child). */
int splats_export(unsigned long long* keys, unsigned* perm, int* children, int* parents,
                  float* node_aabbs);

/* The exact child boxes of every internal node j (Karras numbering): the 12 floats of its 64-byte
 * record -- left child box lo xyz, hi xyz, then the right child's -- copied verbatim
 * (splats_export's node_aabbs are derived: a node's box there is the union of these two).  Needs
 * SPLATS_OPT_EXACT_NODES during the build (ESTATE otherwise), like node_aabbs.
 *   child_boxes  dev, (N-1)*12 float32.  Synchronises.  Parity only. */
int splats_export_child_boxes(float* child_boxes);

/* The records the traversal actually reads, copied verbatim: for every internal node j eight
 * uint32 -- words 0..2: axis x, y, z of the left child box, q_lo | q_hi << 16; words 3..5: the right
 * child's; words 6, 7: left / right link (>= 0: internal node; < 0: the leaf at sorted position
 * link & 0x3ffffff).  The 16-bit codes quantise the exact child boxes (oracle step O7) over the
 * frame [lo - rmax, hi + rmax] (lo / hi: bounds of the splat centres, rmax: the largest radius),
 * lower planes rounded down, upper planes rounded up (S13): a quantised box
 * contains the exact one and the image is unchanged, the records are half the size.
 *   qnodes  dev, (N-1)*8 uint32 (may be NULL)
 *   frame   dev, 7 float32: lo xyz, hi xyz, rmax (may be NULL)
 * Synchronises.  Parity only. */
int splats_export_qnodes(unsigned* qnodes, float* frame);

/* Export the splats themselves in sorted order (dev pointers, may be NULL): sphere N*4
 * float32 (cx, cy, cz, r), rgba N*4 float32; and the scene bounds (min/max of the centres)
 * lo_hi: 6 float32.  Synchronises.  Parity/debug only. */
int splats_export_splats(float* sphere, float* rgba, float* lo_hi);

/* Implementation variants (same results, bit for bit; for A/B measurement).  Takes effect at
 * the next splats_update.
 *   SPLATS_OPT_REFIT: how step a5 (node boxes) is computed.
 *     SPLATS_REFIT_TILED (default): one block per 1024 sorted leaves builds every subtree inside its
 *       tile bottom-up in shared memory (boxes and topology together); the few nodes that span
 *       tiles are finished by a second kernel with range queries on a min/max pyramid.
 *     SPLATS_REFIT_PYRAMID: a bottom-up min/max pyramid over the sorted leaf boxes, Karras'
 *       per-node searches, then every node reads its two child boxes as range queries.
 *     SPLATS_REFIT_ATOMIC: one thread per leaf climbs the tree; the second arrival at a node's
 *       atomic counter forms the union and continues (the classic LBVH refit).
 *   SPLATS_OPT_SORT: how step a3 (order by (code, id)) is computed.
 *     SPLATS_SORT_HYBRID (default): one launch; 3 onesweep passes over the top 24 code bits (4 over the
 *       top 32 above 2^23 splats), after which the array is a sequence of small buckets (a few to a few
 *       dozen keys of a one-sample-per-pixel frame); every bucket is then put in order by (code, id) in
 *       shared memory, window by window, by counting.  A bucket of more than 512 keys makes the launch
 *       fall back to the passes of SPLATS_SORT_HYBRID_LSD from where the array is.
 *     SPLATS_SORT_HYBRID_LSD: one launch; 4 onesweep passes over the top 32 code bits (5 over the top 40
 *       above 2^19 splats), then a check that no two neighbours share them; short runs are fixed up by a
 *       stable insertion sort, longer ones make the same launch redo the sort with all 8 passes.
 *     SPLATS_SORT_LSD8: all 8 passes in one launch (grid barriers between the passes).
 *     SPLATS_SORT_LSD8_LAUNCHES: one launch per pass.
 *   SPLATS_OPT_EXACT_NODES (default 0): after the tiled build, which carries quantised boxes only, the
 *     update also runs the pyramid refit (Karras' per-node searches, exact float32 unions) to store the
 *     exact child boxes (64 bytes per node) for splats_export / splats_export_child_boxes; the
 *     traversal records are untouched.  The other two refit modes always store them.
 *   SPLATS_OPT_PDL (default 1): launch the kernels of splats_update / splats_render as
 *     programmatic dependent launches (each kernel waits on its predecessor at its first
 *     instruction; only the launch latency overlaps).  0 = ordinary stream launches.
 *   SPLATS_OPT_OVERLAP (default 0; needs SPLATS_OPT_PDL): consecutive splats_render* calls that
 *     use the same BVH and write disjoint images do not depend on each other, so up to eight of
 *     them are allowed to execute concurrently: the next render's blocks fill the SMs that the
 *     tail of the previous one leaves idle.  Results are unchanged.  Stream order is kept towards
 *     everything else (updates, other calls of this library, later work of the caller: a render
 *     never completes before the render launched before it), and a
 *     render whose image overlaps one that may still be in flight is serialised.  The one thing
 *     given up: work that the CALLER enqueues between two such render calls is not guaranteed to
 *     be complete before the second render starts writing its image (the render reads nothing
 *     of the caller's, so this only matters if that work writes the same image).
 *     With the option on, the first kernel of a splats_update that directly follows a render
 *     (scene bounds: it reads the caller's depth buffer and touches nothing a render uses) also
 *     starts under that render's tail; the same caveat applies to work the caller enqueues
 *     between the render and the update that writes the frame buffers with programmatic
 *     dependent launches of its own.
 * Errors: EINVAL for an unknown option or value, ESTATE without a context. */
#define SPLATS_OPT_PDL         2
#define SPLATS_OPT_OVERLAP     3
#define SPLATS_OPT_EXACT_NODES 4
#define SPLATS_OPT_REFIT       0
#define SPLATS_REFIT_PYRAMID   0
#define SPLATS_REFIT_ATOMIC    1
#define SPLATS_REFIT_TILED     2
#define SPLATS_OPT_SORT        1
#define SPLATS_SORT_HYBRID         0
#define SPLATS_SORT_LSD8           1
#define SPLATS_SORT_LSD8_LAUNCHES  2
#define SPLATS_SORT_HYBRID_LSD     3
int splats_set_option(int option, int value);

/* How splats_update derives the radius of a splat (takes effect at the next update; SURVEY.md
 * sec. 8(f) row 3).  r_scale of splats_update multiplies all of them.
 *   SPLATS_RADIUS_FOOTPRINT (default; param ignored): half the diagonal of the pixel's footprint
 *     at the splat's view-axis depth (north_star).
 *   SPLATS_RADIUS_CONSTANT: one radius for every splat, r = r_scale * param; the paper sets it
 *     "to half the size of a voxel's diagonal", which the caller passes as param
 *     (object-space length, > 0).
 *   SPLATS_RADIUS_OPACITY: footprint radius * (param + (1 - param) * alpha), param in [0, 1], alpha
 *     the pixel's opacity: a reading of the paper's future-work idea of "varying the radius of
 *     the object space samples according to their opacity"; a splat whose radius
 *     comes out as 0 is kept (it can never be hit).
 * Errors: EINVAL for an unknown mode or a param outside its range, ESTATE without a context. */
#define SPLATS_RADIUS_FOOTPRINT 0
#define SPLATS_RADIUS_CONSTANT  1
#define SPLATS_RADIUS_OPACITY   2
int splats_set_radius(int mode, float param);

/* Per-stage device times, measured with CUDA events recorded on the library's stream around
 * each stage of every update / render issued while profiling is on.  Off by default (the
 * event records cost about a microsecond each, and while it is on the kernels are launched
 * one after the other without programmatic dependent launches).  splats_stage_ms synchronises the stream,
 * returns for each stage the SUM of its durations in milliseconds and how many times it ran
 * since profiling was switched on or since the previous query, and clears the record.
 * stage order: 0 bounds, 1 unproject+morton+compact, 2 sort (all passes), 3 first tree kernel
 * (pyramid mode: gather + leaf boxes + pyramid; atomic mode: gather + hierarchy), 4 the rest of
 * the tree (pyramid mode: hierarchy kernel + node-box kernel, which otherwise runs beside stage
 * 3; atomic mode: refit), 5 render (either query),
 * 6 splats_pack (both launches), 7 splats_render_points (three launches), 8 splats_march.
 * calls may be NULL. */
#define SPLATS_NUM_STAGES 9
int splats_set_profiling(int on);
int splats_stage_ms(float* ms_sum /* host, SPLATS_NUM_STAGES */, unsigned* calls /* host, SPLATS_NUM_STAGES */);

/* Rays actually traced: the sum, over every splats_render* call since splats_create (or since
 * the last call with reset != 0), of the destination pixels that lie in 8x4-pixel tiles inside the
 * screen rectangle of the scene box -- the pixels for which a primary ray was set up and the BVH
 * was walked; every other pixel is written as background without a ray.  Counted
 * by the render kernel.  Synchronises the stream.  Measurement only. */
int splats_traced_pixels(unsigned long long* pixels_host, int reset);

/* How many kernels this library has launched since splats_create. */
unsigned long long splats_launch_count(void);

/* Block until everything enqueued so far has run (kernels and the *_host copies). */
int splats_synchronize(void);

const char* splats_last_error(void);
void splats_destroy(void);

#ifdef __cplusplus
}
#endif
#endif /* SPLATS_H_ */
