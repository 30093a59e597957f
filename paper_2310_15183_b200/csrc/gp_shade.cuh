// gp_shade.cuh — image formation: exit state of every sub-ray -> RGBA8 pixel (the paper's drawing
// kernel; formulas in include/gp.h "image formation").
//
// HBM-bound: one thread per output pixel reads the S*S records of its
// sub-rays — only the first 64-byte half of each: (t, r, theta, phi) and the sector holding status,
// plus the first sector of the disk record — and writes one 4-byte pixel.  Every FP64 operation
// is individually rounded (__dadd_rn / __dmul_rn / __ddiv_rn never contract into FMAs), so the
// bytes are identical to any IEEE-754 evaluation of the same formulas in the same order.
#ifndef GP_SHADE_CUH_
#define GP_SHADE_CUH_

#include "../../include/gp.h"

namespace gp {
#if defined(__CUDACC__)

struct ShadeParams {
  long long W, H, S;
  int mode, disk_overlay;
  double step_rad, hw_rad;      // grid step and half width in radians (host: deg * (pi/180))
  long long tw, th;
  unsigned long long tex_seed;
  double time_period, g_lo, g_hi;
  const gp_ray_record *rays;
  const gp_disk_record *disk;
  unsigned char *rgba;
};

__constant__ double kPalette8[8][3] = {{.85, .25, .25}, {.25, .75, .25}, {.25, .35, .9}, {.9, .8, .2},
                                       {.55, .15, .15}, {.15, .45, .15}, {.15, .2, .6},  {.6, .5, .1}};
__constant__ double kPalette6[6][3] = {{.9, .1, .1}, {.9, .6, .1}, {.8, .9, .1}, {.1, .8, .2}, {.1, .5, .9}, {.6, .1, .9}};

// byte / 255.0, correctly rounded by the host compiler: the same double the IEEE division gives, without
// twelve FP64 divisions per bilinear sample (they made the kernel compute-bound)
__constant__ double kByteOver255[256] = {
    0.0 / 255.0, 1.0 / 255.0, 2.0 / 255.0, 3.0 / 255.0, 4.0 / 255.0, 5.0 / 255.0, 6.0 / 255.0, 7.0 / 255.0,
    8.0 / 255.0, 9.0 / 255.0, 10.0 / 255.0, 11.0 / 255.0, 12.0 / 255.0, 13.0 / 255.0, 14.0 / 255.0, 15.0 / 255.0,
    16.0 / 255.0, 17.0 / 255.0, 18.0 / 255.0, 19.0 / 255.0, 20.0 / 255.0, 21.0 / 255.0, 22.0 / 255.0, 23.0 / 255.0,
    24.0 / 255.0, 25.0 / 255.0, 26.0 / 255.0, 27.0 / 255.0, 28.0 / 255.0, 29.0 / 255.0, 30.0 / 255.0, 31.0 / 255.0,
    32.0 / 255.0, 33.0 / 255.0, 34.0 / 255.0, 35.0 / 255.0, 36.0 / 255.0, 37.0 / 255.0, 38.0 / 255.0, 39.0 / 255.0,
    40.0 / 255.0, 41.0 / 255.0, 42.0 / 255.0, 43.0 / 255.0, 44.0 / 255.0, 45.0 / 255.0, 46.0 / 255.0, 47.0 / 255.0,
    48.0 / 255.0, 49.0 / 255.0, 50.0 / 255.0, 51.0 / 255.0, 52.0 / 255.0, 53.0 / 255.0, 54.0 / 255.0, 55.0 / 255.0,
    56.0 / 255.0, 57.0 / 255.0, 58.0 / 255.0, 59.0 / 255.0, 60.0 / 255.0, 61.0 / 255.0, 62.0 / 255.0, 63.0 / 255.0,
    64.0 / 255.0, 65.0 / 255.0, 66.0 / 255.0, 67.0 / 255.0, 68.0 / 255.0, 69.0 / 255.0, 70.0 / 255.0, 71.0 / 255.0,
    72.0 / 255.0, 73.0 / 255.0, 74.0 / 255.0, 75.0 / 255.0, 76.0 / 255.0, 77.0 / 255.0, 78.0 / 255.0, 79.0 / 255.0,
    80.0 / 255.0, 81.0 / 255.0, 82.0 / 255.0, 83.0 / 255.0, 84.0 / 255.0, 85.0 / 255.0, 86.0 / 255.0, 87.0 / 255.0,
    88.0 / 255.0, 89.0 / 255.0, 90.0 / 255.0, 91.0 / 255.0, 92.0 / 255.0, 93.0 / 255.0, 94.0 / 255.0, 95.0 / 255.0,
    96.0 / 255.0, 97.0 / 255.0, 98.0 / 255.0, 99.0 / 255.0, 100.0 / 255.0, 101.0 / 255.0, 102.0 / 255.0, 103.0 / 255.0,
    104.0 / 255.0, 105.0 / 255.0, 106.0 / 255.0, 107.0 / 255.0, 108.0 / 255.0, 109.0 / 255.0, 110.0 / 255.0, 111.0 / 255.0,
    112.0 / 255.0, 113.0 / 255.0, 114.0 / 255.0, 115.0 / 255.0, 116.0 / 255.0, 117.0 / 255.0, 118.0 / 255.0, 119.0 / 255.0,
    120.0 / 255.0, 121.0 / 255.0, 122.0 / 255.0, 123.0 / 255.0, 124.0 / 255.0, 125.0 / 255.0, 126.0 / 255.0, 127.0 / 255.0,
    128.0 / 255.0, 129.0 / 255.0, 130.0 / 255.0, 131.0 / 255.0, 132.0 / 255.0, 133.0 / 255.0, 134.0 / 255.0, 135.0 / 255.0,
    136.0 / 255.0, 137.0 / 255.0, 138.0 / 255.0, 139.0 / 255.0, 140.0 / 255.0, 141.0 / 255.0, 142.0 / 255.0, 143.0 / 255.0,
    144.0 / 255.0, 145.0 / 255.0, 146.0 / 255.0, 147.0 / 255.0, 148.0 / 255.0, 149.0 / 255.0, 150.0 / 255.0, 151.0 / 255.0,
    152.0 / 255.0, 153.0 / 255.0, 154.0 / 255.0, 155.0 / 255.0, 156.0 / 255.0, 157.0 / 255.0, 158.0 / 255.0, 159.0 / 255.0,
    160.0 / 255.0, 161.0 / 255.0, 162.0 / 255.0, 163.0 / 255.0, 164.0 / 255.0, 165.0 / 255.0, 166.0 / 255.0, 167.0 / 255.0,
    168.0 / 255.0, 169.0 / 255.0, 170.0 / 255.0, 171.0 / 255.0, 172.0 / 255.0, 173.0 / 255.0, 174.0 / 255.0, 175.0 / 255.0,
    176.0 / 255.0, 177.0 / 255.0, 178.0 / 255.0, 179.0 / 255.0, 180.0 / 255.0, 181.0 / 255.0, 182.0 / 255.0, 183.0 / 255.0,
    184.0 / 255.0, 185.0 / 255.0, 186.0 / 255.0, 187.0 / 255.0, 188.0 / 255.0, 189.0 / 255.0, 190.0 / 255.0, 191.0 / 255.0,
    192.0 / 255.0, 193.0 / 255.0, 194.0 / 255.0, 195.0 / 255.0, 196.0 / 255.0, 197.0 / 255.0, 198.0 / 255.0, 199.0 / 255.0,
    200.0 / 255.0, 201.0 / 255.0, 202.0 / 255.0, 203.0 / 255.0, 204.0 / 255.0, 205.0 / 255.0, 206.0 / 255.0, 207.0 / 255.0,
    208.0 / 255.0, 209.0 / 255.0, 210.0 / 255.0, 211.0 / 255.0, 212.0 / 255.0, 213.0 / 255.0, 214.0 / 255.0, 215.0 / 255.0,
    216.0 / 255.0, 217.0 / 255.0, 218.0 / 255.0, 219.0 / 255.0, 220.0 / 255.0, 221.0 / 255.0, 222.0 / 255.0, 223.0 / 255.0,
    224.0 / 255.0, 225.0 / 255.0, 226.0 / 255.0, 227.0 / 255.0, 228.0 / 255.0, 229.0 / 255.0, 230.0 / 255.0, 231.0 / 255.0,
    232.0 / 255.0, 233.0 / 255.0, 234.0 / 255.0, 235.0 / 255.0, 236.0 / 255.0, 237.0 / 255.0, 238.0 / 255.0, 239.0 / 255.0,
    240.0 / 255.0, 241.0 / 255.0, 242.0 / 255.0, 243.0 / 255.0, 244.0 / 255.0, 245.0 / 255.0, 246.0 / 255.0, 247.0 / 255.0,
    248.0 / 255.0, 249.0 / 255.0, 250.0 / 255.0, 251.0 / 255.0, 252.0 / 255.0, 253.0 / 255.0, 254.0 / 255.0, 255.0 / 255.0};

namespace sh {
constexpr double kPi = 3.14159265358979323846;
constexpr double kTwoPi = 2.0 * kPi;
__device__ __forceinline__ double add(double a, double b) { return __dadd_rn(a, b); }
__device__ __forceinline__ double sub(double a, double b) { return __dadd_rn(a, -b); }
__device__ __forceinline__ double mul(double a, double b) { return __dmul_rn(a, b); }
__device__ __forceinline__ double div(double a, double b) { return __ddiv_rn(a, b); }
__device__ __forceinline__ double clamp01(double x) { return x < 0.0 ? 0.0 : (x > 1.0 ? 1.0 : x); }
__device__ __forceinline__ double dist_to_multiple(double x, double step) {
  double k = floor(add(div(x, step), 0.5));
  return fabs(sub(x, mul(k, step)));
}
__device__ __forceinline__ unsigned long long splitmix64(unsigned long long z) {
  z += 0x9E3779B97F4A7C15ULL;
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
  return z ^ (z >> 31);
}
__device__ __forceinline__ void texel(const double *b255, unsigned long long seed, int tw, int i, int j,
                                      double c[3]) {
  unsigned long long h = splitmix64(seed * 0x9E3779B97F4A7C15ULL + (unsigned long long)((long long)j * tw + i));
  c[0] = b255[h & 0xff];
  c[1] = b255[(h >> 8) & 0xff];
  c[2] = b255[(h >> 16) & 0xff];
}
__device__ __forceinline__ double lerp(double a, double x, double b) { return add(a, mul(x, sub(b, a))); }
}  // namespace sh

__device__ __forceinline__ void shade_ray(const ShadeParams &P, const double *b255, unsigned status, double theta, double phi, double t,
                                          double disk_r0, double disk_g0, double rgb[3]) {
  using namespace sh;
  if (P.disk_overlay && !(disk_r0 != disk_r0)) {
    if (disk_g0 < 1.0) {
      double x = clamp01(div(sub(disk_g0, P.g_lo), sub(1.0, P.g_lo)));
      rgb[0] = lerp(0.1, x, 1.0); rgb[1] = lerp(0.2, x, 1.0); rgb[2] = lerp(1.0, x, 1.0);
    } else {
      double x = clamp01(div(sub(disk_g0, 1.0), sub(P.g_hi, 1.0)));
      rgb[0] = lerp(1.0, x, 1.0); rgb[1] = lerp(1.0, x, 0.1); rgb[2] = lerp(1.0, x, 0.1);
    }
    return;
  }
  if (status != GP_RAY_ESCAPED) {
    rgb[0] = 0.0;
    rgb[1] = rgb[2] = (P.mode == 2) ? 1.0 : 0.0;
    return;
  }
  // canonical angles without transcendentals
  double th = sub(theta, mul(kTwoPi, floor(div(theta, kTwoPi))));
  double ph = phi;
  if (th > kPi) {
    th = sub(kTwoPi, th);
    ph = add(ph, kPi);
  }
  ph = sub(ph, mul(kTwoPi, floor(div(ph, kTwoPi))));
  if (P.mode == 0) {
    long long q = (long long)floor(div(ph, mul(0.5, kPi)));
    if (q > 3) q = 3;
    long long idx = ((th >= mul(0.5, kPi)) ? 4 : 0) + q;
    bool line = dist_to_multiple(th, P.step_rad) < P.hw_rad || dist_to_multiple(ph, P.step_rad) < P.hw_rad;
    for (int k = 0; k < 3; ++k) rgb[k] = line ? 0.05 : kPalette8[idx][k];
  } else if (P.mode == 1) {
    const int tw = (int)P.tw, thh = (int)P.th;   // validated <= 2^30 on the host; 32-bit index arithmetic
    double u = sub(mul(div(ph, kTwoPi), (double)tw), 0.5);
    double v = sub(mul(div(th, kPi), (double)thh), 0.5);
    double fu = floor(u), fv = floor(v);
    double au = sub(u, fu), av = sub(v, fv);
    int i0 = (int)fu, j0 = (int)fv;               // u in [-0.5, tw - 0.5): i0 in [-1, tw - 1]
    int i1 = i0 + 1, j1 = j0 + 1;
    i0 = i0 < 0 ? i0 + tw : i0;
    i1 = i1 >= tw ? i1 - tw : i1;
    j0 = j0 < 0 ? 0 : (j0 > thh - 1 ? thh - 1 : j0);
    j1 = j1 < 0 ? 0 : (j1 > thh - 1 ? thh - 1 : j1);
    double c00[3], c10[3], c01[3], c11[3];
    texel(b255, P.tex_seed, tw, i0, j0, c00);
    texel(b255, P.tex_seed, tw, i1, j0, c10);
    texel(b255, P.tex_seed, tw, i0, j1, c01);
    texel(b255, P.tex_seed, tw, i1, j1, c11);
    for (int k = 0; k < 3; ++k) {
      double top = lerp(c00[k], au, c10[k]);
      double bot = lerp(c01[k], au, c11[k]);
      rgb[k] = lerp(top, av, bot);
    }
  } else {
    long long band = (long long)floor(div(fabs(t), P.time_period));
    long long idx = band % 6;
    for (int k = 0; k < 3; ++k) rgb[k] = kPalette6[idx][k];
  }
}

// One thread per output pixel; consecutive threads take consecutive pixels of a row, so for S = 1 a
// warp reads 32 consecutive records (the two 32-byte sectors it needs of each) and writes 128
// contiguous bytes.
__global__ void k_shade(const __grid_constant__ ShadeParams P) {
  // the byte/255 table goes to shared memory: lanes index it with unrelated bytes, which constant
  // memory would serialise (measured: 0.258 ms from __constant__ against 0.166 ms with 12 divisions)
  __shared__ double b255[256];
  for (int k = threadIdx.x; k < 256; k += blockDim.x) b255[k] = kByteOver255[k];
  __syncthreads();
  const long long pix = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (pix >= P.W * P.H) return;
  const long long j = pix / P.W, i = pix - j * P.W;
  double sum[3] = {0.0, 0.0, 0.0};
  const double qnan = __longlong_as_double(0x7ff8000000000000LL);
  for (long long sj = 0; sj < P.S; ++sj)
    for (long long si = 0; si < P.S; ++si) {
      const long long ray = (j * P.S + sj) * P.W * P.S + (i * P.S + si);
      // the first 64-byte half of the record: (t, r | theta, phi | lambda, status..) as three 128-bit loads
      // with a 64-byte L2 prefetch-size hint, so that the second half is not pulled in with it
      const char *rec = reinterpret_cast<const char *>(P.rays + ray);
#pragma nv_diag_suppress 550
      double t, r_unused, th_raw, ph_raw;
      unsigned b0, b1, status, b3;
#pragma nv_diag_default 550
      asm volatile("ld.global.nc.L2::64B.v2.f64 {%0, %1}, [%2];" : "=d"(t), "=d"(r_unused) : "l"(rec));
      asm volatile("ld.global.nc.L2::64B.v2.f64 {%0, %1}, [%2];" : "=d"(th_raw), "=d"(ph_raw) : "l"(rec + 16));
      asm volatile("ld.global.nc.L2::64B.v4.u32 {%0, %1, %2, %3}, [%4];"
                   : "=r"(b0), "=r"(b1), "=r"(status), "=r"(b3)
                   : "l"(rec + 32));
      (void)r_unused; (void)b0; (void)b1; (void)b3;
      double dr = qnan, dg = qnan;
      if (P.disk_overlay) {
        dr = __ldg(&P.disk[ray].r_cross[0]);
        dg = __ldg(&P.disk[ray].g[0]);
      }
      double rgb[3];
      shade_ray(P, b255, status, th_raw, ph_raw, t, dr, dg, rgb);
      for (int k = 0; k < 3; ++k) sum[k] = sh::add(sum[k], rgb[k]);
    }
  const double inv = sh::div(1.0, (double)(P.S * P.S));
  unsigned out = 0xff000000u;
  for (int k = 0; k < 3; ++k) {
    double q = floor(sh::add(sh::mul(255.0, sh::mul(sum[k], inv)), 0.5));
    unsigned byte = (unsigned)(q < 0.0 ? 0.0 : (q > 255.0 ? 255.0 : q));
    out |= byte << (8 * k);
  }
  reinterpret_cast<unsigned *>(P.rgba)[pix] = out;
}

#endif  // __CUDACC__
}  // namespace gp
#endif
