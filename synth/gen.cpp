// synth/gen.cpp -- seeded synthetic *input* generator (the "server step").
//
// This module is neither the oracle nor the product: it only manufactures the
// 2.5D frames (premultiplied RGBA + one depth per pixel) that BOTH the CPU
// oracle and the CUDA path consume.  It holds none of the client method's
// arithmetic (no splats, no Morton codes, no BVH, no sphere tests).
//
// What it stands in for: the paper's server-side volume ray marcher
// (sec. 4.1 "we render the volume using a ray marcher that employs
// one of the heuristics ... to estimate which depth value represents the volume
// best"; sec. 4.2 "writes out colors and t values to an off-screen
// buffer") run on the paper's unnamed data set, which is not available.  The
// recipe is BASELINE.json `configs` + SURVEY.md sec. 8(d); see DESIGN.md
// "Input recipe".
//
// Everything is computed in double precision and rounded once to float32 on
// output.  Threads (OpenMP) only split independent voxels / pixels, so the
// output does not depend on the thread count.
#include <cmath>
#include <cstdint>
#include <cstdlib>
#include <cstring>
#include <vector>

namespace {

// splitmix64: i-th output (i = 0,1,...) of the stream seeded with `seed`.
inline uint64_t splitmix64_at(uint64_t seed, uint64_t i) {
  uint64_t z = seed + (i + 1) * 0x9E3779B97F4A7C15ull;
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
  return z ^ (z >> 31);
}
inline double u01(uint64_t r) { return (double)(r >> 11) * (1.0 / 9007199254740992.0); }

struct Cam {
  double eye[3], right[3], up[3], fwd[3], tanh;
};

inline double clamp01(double v) { return v < 0.0 ? 0.0 : (v > 1.0 ? 1.0 : v); }

// Transfer function: two opacity tents (half-width 0.05): 0.8 at iso 0.35 and
// 0.95 at iso 0.7 (BASELINE.json configs[0]), zero elsewhere; each tent has a
// fixed base colour.
inline void transfer(double d, double& a, double rgb[3]) {
  const double hw = 0.05;
  double w1 = 1.0 - std::fabs(d - 0.35) / hw;
  double w2 = 1.0 - std::fabs(d - 0.70) / hw;
  if (w1 < 0.0) w1 = 0.0;
  if (w2 < 0.0) w2 = 0.0;
  a = 0.8 * w1 + 0.95 * w2;
  if (w1 > 0.0) { rgb[0] = 0.95; rgb[1] = 0.55; rgb[2] = 0.15; }
  else          { rgb[0] = 0.25; rgb[1] = 0.60; rgb[2] = 0.95; }
}

}  // namespace

extern "C" {

// Fill `vol` (n*n*n float32, x fastest) with clamp(sum of n_gauss anisotropic
// Gaussians [+ uniform noise in [-noise_amp, noise_amp]], 0, 1), sampled at voxel
// centres ((i+.5)/n).  Draw order of the splitmix64 stream seeded with `seed`:
// per Gaussian (cx,cy,cz in [0.2,0.8]; sx,sy,sz in [0.05,0.15]), then one draw
// per voxel in memory order for the noise.
void synth_volume(float* vol, int n, int n_gauss, double noise_amp, uint64_t seed) {
  std::vector<double> ex((size_t)n_gauss * n), ey((size_t)n_gauss * n), ez((size_t)n_gauss * n);
  for (int g = 0; g < n_gauss; ++g) {
    double c[3], s[3];
    for (int k = 0; k < 3; ++k) c[k] = 0.2 + 0.6 * u01(splitmix64_at(seed, (uint64_t)g * 6 + k));
    for (int k = 0; k < 3; ++k) s[k] = 0.05 + 0.10 * u01(splitmix64_at(seed, (uint64_t)g * 6 + 3 + k));
    for (int i = 0; i < n; ++i) {
      double x = (i + 0.5) / n;
      double qx = (x - c[0]) / s[0], qy = (x - c[1]) / s[1], qz = (x - c[2]) / s[2];
      ex[(size_t)g * n + i] = std::exp(-0.5 * qx * qx);
      ey[(size_t)g * n + i] = std::exp(-0.5 * qy * qy);
      ez[(size_t)g * n + i] = std::exp(-0.5 * qz * qz);
    }
  }
  const uint64_t noise_base = (uint64_t)n_gauss * 6;
#pragma omp parallel for schedule(static)
  for (int k = 0; k < n; ++k) {
    std::vector<double> yz(n_gauss);
    std::vector<double> row(n);
    for (int j = 0; j < n; ++j) {
      for (int g = 0; g < n_gauss; ++g) yz[g] = ey[(size_t)g * n + j] * ez[(size_t)g * n + k];
      for (int i = 0; i < n; ++i) row[i] = 0.0;
      for (int g = 0; g < n_gauss; ++g) {
        const double w = yz[g];
        if (w < 1e-30) continue;
        const double* e = &ex[(size_t)g * n];
        for (int i = 0; i < n; ++i) row[i] += w * e[i];
      }
      size_t base = ((size_t)k * n + j) * n;
      for (int i = 0; i < n; ++i) {
        double d = row[i];
        if (noise_amp > 0.0) d += noise_amp * (2.0 * u01(splitmix64_at(seed, noise_base + base + i)) - 1.0);
        vol[base + i] = (float)clamp01(d);
      }
    }
  }
}

// Server pass: perspective ray march of `vol` (unit cube [0,1]^3) at 0.5-voxel
// steps.  cam13 = eye, right, up, fwd, tan(fovy/2) (13 float32 values, the same
// struct the client is given).  Per pixel (row 0 = top, pixel centres at +0.5):
//   color[p] = premultiplied front-to-back composite (float32 x4),
//   depth[p] = ray parameter t (unit-length direction) of the first sample at which
//              the accumulated alpha is >= 0.5; 0 if it never gets there (dropped).
// The march stops once accumulated alpha >= 0.999.
void synth_march(const float* vol, int n, const float* cam13, int W, int H,
                 float* color, float* depth) {
  Cam c;
  for (int k = 0; k < 3; ++k) {
    c.eye[k] = cam13[k]; c.right[k] = cam13[3 + k]; c.up[k] = cam13[6 + k]; c.fwd[k] = cam13[9 + k];
  }
  c.tanh = cam13[12];
  const double step = 0.5 / n;
  const double aspect = (double)W / (double)H;
#pragma omp parallel for schedule(dynamic, 4)
  for (int y = 0; y < H; ++y) {
    for (int x = 0; x < W; ++x) {
      const size_t p = (size_t)y * W + x;
      double u = ((2.0 * (x + 0.5) - W) / W) * c.tanh * aspect;
      double v = ((H - 2.0 * (y + 0.5)) / H) * c.tanh;
      double d[3];
      for (int k = 0; k < 3; ++k) d[k] = c.fwd[k] + u * c.right[k] + v * c.up[k];
      double len = std::sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
      for (int k = 0; k < 3; ++k) d[k] /= len;
      // ray / unit-cube slabs
      double t0 = 0.0, t1 = 1e300;
      bool miss = false;
      for (int k = 0; k < 3; ++k) {
        if (std::fabs(d[k]) < 1e-300) {
          if (c.eye[k] < 0.0 || c.eye[k] > 1.0) miss = true;
          continue;
        }
        double a = (0.0 - c.eye[k]) / d[k], b = (1.0 - c.eye[k]) / d[k];
        if (a > b) { double s = a; a = b; b = s; }
        if (a > t0) t0 = a;
        if (b < t1) t1 = b;
      }
      double C[3] = {0, 0, 0}, A = 0.0, tdepth = 0.0;
      if (!miss && t0 < t1) {
        for (long s = 0;; ++s) {
          double t = t0 + (s + 0.5) * step;
          if (t >= t1) break;
          double P[3];
          for (int k = 0; k < 3; ++k) P[k] = c.eye[k] + t * d[k];
          // trilinear, voxel-centred, clamp to edge
          double g[3]; int i0[3], i1[3]; double f[3];
          for (int k = 0; k < 3; ++k) {
            g[k] = P[k] * n - 0.5;
            double fl = std::floor(g[k]);
            f[k] = g[k] - fl;
            int a = (int)fl, b = a + 1;
            if (a < 0) a = 0; if (a > n - 1) a = n - 1;
            if (b < 0) b = 0; if (b > n - 1) b = n - 1;
            i0[k] = a; i1[k] = b;
          }
          auto V = [&](int i, int j, int k) -> double { return vol[((size_t)k * n + j) * n + i]; };
          double c00 = V(i0[0], i0[1], i0[2]) * (1 - f[0]) + V(i1[0], i0[1], i0[2]) * f[0];
          double c10 = V(i0[0], i1[1], i0[2]) * (1 - f[0]) + V(i1[0], i1[1], i0[2]) * f[0];
          double c01 = V(i0[0], i0[1], i1[2]) * (1 - f[0]) + V(i1[0], i0[1], i1[2]) * f[0];
          double c11 = V(i0[0], i1[1], i1[2]) * (1 - f[0]) + V(i1[0], i1[1], i1[2]) * f[0];
          double c0 = c00 * (1 - f[1]) + c10 * f[1], c1 = c01 * (1 - f[1]) + c11 * f[1];
          double dens = c0 * (1 - f[2]) + c1 * f[2];
          double a, rgb[3];
          transfer(dens, a, rgb);
          if (a > 0.0) {
            double T = 1.0 - A;
            for (int k = 0; k < 3; ++k) C[k] += T * a * rgb[k] * (0.55 + 0.45 * clamp01(P[k]));
            A += T * a;
            if (tdepth == 0.0 && A >= 0.5) tdepth = t;
            if (A >= 0.999) break;
          }
        }
      }
      color[4 * p + 0] = (float)C[0]; color[4 * p + 1] = (float)C[1];
      color[4 * p + 2] = (float)C[2]; color[4 * p + 3] = (float)A;
      depth[p] = (float)tdepth;
    }
  }
}

}  // extern "C"
