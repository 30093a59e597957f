// gp_shade_oracle.cpp — TEST INFRASTRUCTURE, not the product.
//
// Plain scalar reference for the image-formation step (the paper's "drawing script" kernel,
// PAPER.md L404, L422, L430, L446, L735): exit state of every sub-ray -> RGBA8 pixel.  Written from
// the formulas stated in include/gp.h (section "image formation") and DESIGN.md section 10; shares
// nothing with the CUDA library.  Built with -ffp-contract=off so that every operation is rounded
// on its own; the result is defined bit for bit.
//
// Pins (tests/test_oracle_shade_pins.py): SplitMix64 test vector; canonical angles against
// acos(cos)/atan2; hand-computed palette, grid-line and band cases; bilinear filter at texel
// centres and against a numpy gather; g = g_lo, 1, g_hi colours; supersampling of identical
// sub-rays; all-captured image.
#include <cmath>
#include <cstdint>
#include <cstring>

namespace {

const double kPi = 3.14159265358979323846;
const double kTwoPi = 2.0 * kPi;

const double kPalette8[8][3] = {{.85, .25, .25}, {.25, .75, .25}, {.25, .35, .9}, {.9, .8, .2},
                                {.55, .15, .15}, {.15, .45, .15}, {.15, .2, .6},  {.6, .5, .1}};
const double kPalette6[6][3] = {{.9, .1, .1}, {.9, .6, .1}, {.8, .9, .1}, {.1, .8, .2}, {.1, .5, .9}, {.6, .1, .9}};

uint64_t splitmix64(uint64_t z) {
  z += 0x9E3779B97F4A7C15ULL;
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
  return z ^ (z >> 31);
}

void texel(uint64_t seed, int64_t tw, int64_t i, int64_t j, double c[3]) {
  uint64_t h = splitmix64(seed * 0x9E3779B97F4A7C15ULL + (uint64_t)(j * tw + i));
  c[0] = (double)(h & 0xff) / 255.0;
  c[1] = (double)((h >> 8) & 0xff) / 255.0;
  c[2] = (double)((h >> 16) & 0xff) / 255.0;
}

double clamp01(double x) { return x < 0.0 ? 0.0 : (x > 1.0 ? 1.0 : x); }

// distance of x to the nearest multiple of step
double dist_to_multiple(double x, double step) {
  double k = std::floor(x / step + 0.5);
  return std::fabs(x - k * step);
}

}  // namespace

extern "C" {

struct orc_shade_cfg {
  int64_t width, height, supersample, mode;
  double grid_step_deg, grid_half_width_deg;
  int64_t tex_width, tex_height;
  uint64_t tex_seed;
  double time_period;
  int64_t disk_overlay;
  double g_lo, g_hi;
};

uint64_t orc_splitmix64(uint64_t z) { return splitmix64(z); }

// canonical angles of a raw exit direction: out2 = (theta in [0, pi], phi in [0, 2 pi))
void orc_canonical_angles(double theta, double phi, double *out2) {
  double th = theta - kTwoPi * std::floor(theta / kTwoPi);
  double ph = phi;
  if (th > kPi) {
    th = kTwoPi - th;
    ph = ph + kPi;
  }
  ph = ph - kTwoPi * std::floor(ph / kTwoPi);
  out2[0] = th;
  out2[1] = ph;
}

// colour of one sub-ray; disk_r0 / disk_g0 = first recorded crossing (NaN when none / no disk buffer)
void orc_shade_ray(const orc_shade_cfg *cfg, int64_t status, double theta, double phi, double t, double disk_r0,
                   double disk_g0, double rgb[3]) {
  if (cfg->disk_overlay && !std::isnan(disk_r0)) {
    const double blue[3] = {0.1, 0.2, 1.0}, red[3] = {1.0, 0.1, 0.1};
    if (disk_g0 < 1.0) {
      double x = clamp01((disk_g0 - cfg->g_lo) / (1.0 - cfg->g_lo));
      for (int k = 0; k < 3; ++k) rgb[k] = blue[k] + x * (1.0 - blue[k]);
    } else {
      double x = clamp01((disk_g0 - 1.0) / (cfg->g_hi - 1.0));
      for (int k = 0; k < 3; ++k) rgb[k] = 1.0 + x * (red[k] - 1.0);
    }
    return;
  }
  if (status != 0) {
    rgb[0] = 0.0;
    rgb[1] = rgb[2] = (cfg->mode == 2) ? 1.0 : 0.0;
    return;
  }
  double ang[2];
  orc_canonical_angles(theta, phi, ang);
  const double th = ang[0], ph = ang[1];
  if (cfg->mode == 0) {
    int64_t q = (int64_t)std::floor(ph / (0.5 * kPi));
    if (q > 3) q = 3;
    int64_t idx = ((th >= 0.5 * kPi) ? 4 : 0) + q;
    const double step = cfg->grid_step_deg * (kPi / 180.0), hw = cfg->grid_half_width_deg * (kPi / 180.0);
    bool line = dist_to_multiple(th, step) < hw || dist_to_multiple(ph, step) < hw;
    for (int k = 0; k < 3; ++k) rgb[k] = line ? 0.05 : kPalette8[idx][k];
  } else if (cfg->mode == 1) {
    const int64_t tw = cfg->tex_width, thh = cfg->tex_height;
    double u = ph / kTwoPi * (double)tw - 0.5;
    double v = th / kPi * (double)thh - 0.5;
    double fu = std::floor(u), fv = std::floor(v);
    double au = u - fu, av = v - fv;
    int64_t i0 = (int64_t)fu, j0 = (int64_t)fv;
    int64_t i1 = i0 + 1, j1 = j0 + 1;
    i0 = ((i0 % tw) + tw) % tw;
    i1 = ((i1 % tw) + tw) % tw;
    if (j0 < 0) j0 = 0;
    if (j0 > thh - 1) j0 = thh - 1;
    if (j1 < 0) j1 = 0;
    if (j1 > thh - 1) j1 = thh - 1;
    double c00[3], c10[3], c01[3], c11[3];
    texel(cfg->tex_seed, tw, i0, j0, c00);
    texel(cfg->tex_seed, tw, i1, j0, c10);
    texel(cfg->tex_seed, tw, i0, j1, c01);
    texel(cfg->tex_seed, tw, i1, j1, c11);
    for (int k = 0; k < 3; ++k) {
      double top = c00[k] + au * (c10[k] - c00[k]);
      double bot = c01[k] + au * (c11[k] - c01[k]);
      rgb[k] = top + av * (bot - top);
    }
  } else {
    int64_t band = (int64_t)std::floor(std::fabs(t) / cfg->time_period);
    int64_t idx = band % 6;
    for (int k = 0; k < 3; ++k) rgb[k] = kPalette6[idx][k];
  }
}

// whole image.  rays: n records in the CUDA library's 128-byte layout is NOT assumed: the caller
// passes plain arrays (status, theta, phi, t, disk_r0, disk_g0) of n = W*H*S*S entries.
int orc_shade(const orc_shade_cfg *cfg, const int64_t *status, const double *theta, const double *phi,
              const double *t, const double *disk_r0, const double *disk_g0, uint8_t *rgba) {
  const int64_t W = cfg->width, H = cfg->height, S = cfg->supersample;
  if (W <= 0 || H <= 0 || S <= 0 || cfg->mode < 0 || cfg->mode > 2) return -2;
  const double inv = 1.0 / (double)(S * S);
  const double nan = std::nan("");
  for (int64_t j = 0; j < H; ++j)
    for (int64_t i = 0; i < W; ++i) {
      double sum[3] = {0.0, 0.0, 0.0};
      for (int64_t sj = 0; sj < S; ++sj)
        for (int64_t si = 0; si < S; ++si) {
          int64_t ray = (j * S + sj) * W * S + (i * S + si);
          double rgb[3];
          orc_shade_ray(cfg, status[ray], theta[ray], phi[ray], t[ray], disk_r0 ? disk_r0[ray] : nan,
                        disk_g0 ? disk_g0[ray] : nan, rgb);
          for (int k = 0; k < 3; ++k) sum[k] = sum[k] + rgb[k];
        }
      uint8_t *px = rgba + 4 * (j * W + i);
      for (int k = 0; k < 3; ++k) {
        double q = std::floor(255.0 * (sum[k] * inv) + 0.5);
        px[k] = (uint8_t)(q < 0.0 ? 0.0 : (q > 255.0 ? 255.0 : q));
      }
      px[3] = 255;
    }
  return 0;
}

}  // extern "C"
