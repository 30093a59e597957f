// gp_api.cu — C-ABI of libgp.so (include/gp.h): synchronous validation, per-launch constants
// derived on the host in FP64, asynchronous launches on the caller's stream.
// There is no CPU path: every step of the method runs in the kernels of gp_trace*.cuh.
#include <cuda_runtime.h>
#include <math.h>
#include <stddef.h>
#include <stdio.h>
#include <string.h>

#include <mutex>

#include "../../include/gp.h"
#include "gp_trace.cuh"
#include "gp_shade.cuh"
#include "gp_orbits.cuh"

static_assert(sizeof(gp_ray_record) == 128, "gp_ray_record must be 128 bytes");
static_assert(offsetof(gp_ray_record, status) == 40 && offsetof(gp_ray_record, p_t) == 64 &&
                  offsetof(gp_ray_record, n_rhs) == 124,
              "gp_ray_record layout (gp_trace.cuh store_record and gp_shade.cuh read it by offset)");
static_assert(sizeof(gp_disk_record) == 48, "gp_disk_record must be 48 bytes");

namespace {

using namespace gp;

thread_local char g_cuda_msg[256] = "";

int cuda_fail(cudaError_t e) {
  snprintf(g_cuda_msg, sizeof(g_cuda_msg), "%s: %s", cudaGetErrorName(e), cudaGetErrorString(e));
  return GP_E_CUDA;
}
#define GP_CUDA(call)                          \
  do {                                         \
    cudaError_t e__ = (call);                  \
    if (e__ != cudaSuccess) return cuda_fail(e__); \
  } while (0)

// ---- validation + constants -------------------------------------------------------------------
int make_metric(int metric_id, const gp_metric_params *m, MetricConst *mc) {
  if (!m) return GP_E_NULL;
  if (metric_id < GP_SCHWARZSCHILD || metric_id > GP_MANKO_NOVIKOV) return GP_E_BAD_METRIC;
  memset(mc, 0, sizeof(*mc));
  double M = m->M, a = m->a, q = m->q;
  if (!isfinite(M) || !isfinite(a) || !isfinite(q)) return GP_E_BAD_PARAM;
  if (metric_id == GP_SCHWARZSCHILD) {
    if (!(M >= 0.0)) return GP_E_BAD_PARAM;  // M = 0: flat space
    a = 0.0;
    q = 0.0;
  } else {
    if (!(M > 0.0) || !(fabs(a) < M)) return GP_E_BAD_PARAM;
    if (metric_id == GP_MANKO_NOVIKOV && a == 0.0) return GP_E_BAD_PARAM;  // eq 23 divides by S/M
    if (metric_id == GP_KERR) q = 0.0;
  }
  mc->M = M;
  mc->a = a;
  mc->q = q;
  mc->a2 = a * a;
  mc->m2M = -2.0 * M;
  mc->r_horizon = (metric_id == GP_SCHWARZSCHILD) ? 2.0 * M : M + sqrt(M * M - a * a);
  if (metric_id == GP_MANKO_NOVIKOV) {
    double al = (-M + sqrt(M * M - a * a)) / a;          // eq 23
    double k = M * (1.0 - al * al) / (1.0 + al * al);    // eq 24
    mc->mn_alpha = al;
    mc->mn_k = k;
    mc->mn_inv_k = 1.0 / k;
    mc->mn_beta = q * M * M * M / (k * k * k);           // eq 25
    mc->mn_w0 = 4.0 * k * al / (1.0 - al * al);
    mc->mn_e0 = k * k / ((1.0 - al * al) * (1.0 - al * al));
  }
  return GP_OK;
}

double isco_prograde(int metric_id, const MetricConst &mc) {
  if (metric_id == GP_MANKO_NOVIKOV) return nan("");
  double M = mc.M;
  double as = (M > 0.0) ? mc.a / M : 0.0;
  double Z1 = 1.0 + cbrt(1.0 - as * as) * (cbrt(1.0 + as) + cbrt(1.0 - as));
  double Z2 = sqrt(3.0 * as * as + Z1 * Z1);
  return M * (3.0 + Z2 - sqrt((3.0 - Z1) * (3.0 + Z1 + 2.0 * Z2)));
}

int make_camera(int metric_id, const MetricConst &mc, const gp_camera *c, double eps_capture, CameraConst *cc) {
  if (!c) return GP_E_NULL;
  if (c->width <= 0 || c->height <= 0 || c->supersample <= 0) return GP_E_BAD_PARAM;
  if (c->projection != 0 && c->projection != 1) return GP_E_UNSUPPORTED;
  if (c->projection == 1 && !(c->focal_2f_over_d >= 0.0 && isfinite(c->focal_2f_over_d))) return GP_E_BAD_PARAM;
  if (!(c->alpha_max > c->alpha_min) || !(c->beta_max > c->beta_min)) return GP_E_BAD_PARAM;
  if (!isfinite(c->alpha_min) || !isfinite(c->alpha_max) || !isfinite(c->beta_min) || !isfinite(c->beta_max))
    return GP_E_BAD_PARAM;
  if (!(c->theta_obs > 0.0) || !(c->theta_obs < 3.14159265358979323846)) return GP_E_BAD_PARAM;
  if (!isfinite(c->r_obs) || !isfinite(c->phi_obs)) return GP_E_BAD_PARAM;
  if (!(c->r_obs > mc.r_horizon * (1.0 + eps_capture)) || !(c->r_obs > 0.0)) return GP_E_BAD_PARAM;
  if (!(c->jitter_amp_px >= 0.0) || !isfinite(c->jitter_amp_px) || !isfinite(c->shift_x_px) ||
      !isfinite(c->shift_y_px))
    return GP_E_BAD_PARAM;
  const long long S = c->supersample;
  const long long Wt = (long long)c->width * S, Ht = (long long)c->height * S;
  const long long total = Wt * Ht;
  if (c->ray_count < 0 || c->ray_begin < 0 || c->ray_stride < 1) return GP_E_BAD_PARAM;
  if (c->ray_count > 0) {
    if (c->ray_begin >= total) return GP_E_BAD_PARAM;
    if ((c->ray_count - 1) > (total - 1 - c->ray_begin) / c->ray_stride) return GP_E_BAD_PARAM;
  }
  memset(cc, 0, sizeof(*cc));
  cc->alpha_min = c->alpha_min;
  cc->beta_min = c->beta_min;
  cc->dalpha = (c->alpha_max - c->alpha_min) / (double)c->width;
  cc->dbeta = (c->beta_max - c->beta_min) / (double)c->height;
  cc->supersample_d = (double)S;
  cc->jitter_amp_px = c->jitter_amp_px;
  cc->shift_x_px = c->shift_x_px;
  cc->shift_y_px = c->shift_y_px;
  cc->jitter_seed = c->jitter_seed;
  cc->Wt = Wt;
  cc->inv_Wt = 1.0 / (double)Wt;
  cc->inv_S = ((S & (S - 1)) == 0) ? 1.0 / (double)S : 0.0;
  cc->ray_begin = c->ray_begin;
  cc->ray_count = c->ray_count;
  cc->ray_stride = c->ray_stride;
  cc->r_obs = c->r_obs;
  cc->theta_obs = c->theta_obs;
  cc->phi_obs = c->phi_obs;
  cc->projection = c->projection;
  cc->metric_id = metric_id;
  cc->k2 = c->focal_2f_over_d;
  cc->a_cam = (metric_id == GP_SCHWARZSCHILD) ? 0.0 : mc.a;
  {
    const double so = sin(c->theta_obs), co = cos(c->theta_obs), sp = sin(c->phi_obs), cp = cos(c->phi_obs);
    cc->chat[0] = so * cp; cc->chat[1] = so * sp; cc->chat[2] = co;
    cc->eph[0] = -sp; cc->eph[1] = cp; cc->eph[2] = 0.0;
    cc->eup[0] = -co * cp; cc->eup[1] = -co * sp; cc->eup[2] = so;
  }
  // observer's ZAMO tetrad from the covariant metric of the selected spacetime (reading R12)
  double g[5];
  metric_cov(metric_id, mc, c->r_obs, c->theta_obs, g);
  double Omega = -g[1] / g[2];
  double lapse2 = -(g[0] + Omega * g[1]);
  if (!(lapse2 > 0.0) || !(g[2] > 0.0) || !(g[3] > 0.0) || !(g[4] > 0.0)) return GP_E_BAD_PARAM;
  cc->Omega = Omega;
  cc->inv_zeta = sqrt(lapse2);
  cc->sq_grr = sqrt(g[3]);
  cc->sq_gthth = sqrt(g[4]);
  cc->sq_gpp = sqrt(g[2]);
  return GP_OK;
}

int make_params(int metric_id, const gp_metric_params *m, const gp_camera *cam, const gp_integrator_cfg *cfg,
                TraceParams *P) {
  if (!m || !cam || !cfg) return GP_E_NULL;
  memset(P, 0, sizeof(*P));
  int rc = make_metric(metric_id, m, &P->mc);
  if (rc) return rc;
  if (cfg->precision < 0 || cfg->precision > 2) return GP_E_UNSUPPORTED;
  if (cfg->scheme < 0 || cfg->scheme > 2) return GP_E_BAD_PARAM;
  // precision 2 (FP32 equations, FP64 state): every scheme; with the adaptive scheme the tolerances must
  // stay above the noise of an FP32 evaluation of the equations in the error estimate (gp.h)
  if (cfg->precision == 2 && cfg->scheme == 2 && (!(cfg->rtol >= 1e-7) || !(cfg->atol >= 1e-7))) return GP_E_BAD_PARAM;
  // the single-precision variant exists for the fixed-step schemes only: a 1e-10 tolerance has no
  // meaning in FP32 arithmetic
  if (cfg->precision == 1 && cfg->scheme == 2) return GP_E_UNSUPPORTED;
  if (!(cfg->eps_capture >= 0.0) || !isfinite(cfg->eps_capture)) return GP_E_BAD_PARAM;
  rc = make_camera(metric_id, P->mc, cam, cfg->eps_capture, &P->cc);
  if (rc) return rc;
  if (cfg->max_steps < 0 || cfg->max_steps > 500000000LL) return GP_E_BAD_PARAM;
  if (!(cfg->r_escape > cam->r_obs) || !isfinite(cfg->r_escape)) return GP_E_BAD_PARAM;
  if (cam->projection == 1) {
    // every start point of the flat screen must lie inside the escape sphere: r <= |X| and the
    // farthest point is a window corner
    double am = fmax(fabs(cam->alpha_min), fabs(cam->alpha_max)), bm = fmax(fabs(cam->beta_min), fabs(cam->beta_max));
    double pad = (cam->jitter_amp_px + fabs(cam->shift_x_px) + fabs(cam->shift_y_px) + 1.0);
    am += pad * (cam->alpha_max - cam->alpha_min) / cam->width;
    bm += pad * (cam->beta_max - cam->beta_min) / cam->height;
    if (!(cfg->r_escape > sqrt(cam->r_obs * cam->r_obs + am * am + bm * bm))) return GP_E_BAD_PARAM;
  }
  if (cfg->scheme == 0 && !(cfg->h > 0.0 && isfinite(cfg->h))) return GP_E_BAD_PARAM;
  if (cfg->scheme == 1 && !(cfg->h_rel > 0.0 && isfinite(cfg->h_rel))) return GP_E_BAD_PARAM;
  if (cfg->scheme == 2) {
    if (!(cfg->rtol > 0.0) || !(cfg->atol >= 0.0) || !(cfg->h_cap_rel > 0.0)) return GP_E_BAD_PARAM;
    if (!isfinite(cfg->rtol) || !isfinite(cfg->atol) || !isfinite(cfg->h_cap_rel)) return GP_E_BAD_PARAM;
  }
  if (cfg->max_crossings < 0 || cfg->max_crossings > 3) return GP_E_BAD_PARAM;
  if (cfg->segment_steps < -1) return GP_E_BAD_PARAM;
  // a Manko-Novikov disk needs an explicit inner radius: there is no ISCO formula for that metric
  if (cfg->max_crossings > 0 && metric_id == GP_MANKO_NOVIKOV && !(cfg->disk_r_in > 0.0)) return GP_E_BAD_PARAM;
  if (isnan(cfg->lambda_max)) return GP_E_BAD_PARAM;
  // solid ring (gp.h): replaces the thin disk, located hits exist for the adaptive scheme
  if (!(cfg->ring_half_angle >= 0.0) || !(cfg->ring_half_angle < 1.5)) return GP_E_BAD_PARAM;
  const bool ring = cfg->ring_half_angle > 0.0;
  if (ring && cfg->max_crossings > 0) return GP_E_UNSUPPORTED;
  if (ring && metric_id == GP_MANKO_NOVIKOV && !(cfg->disk_r_in > 0.0)) return GP_E_BAD_PARAM;
  P->scheme = cfg->scheme;
  P->precision = cfg->precision;
  P->max_crossings = cfg->max_crossings;
  P->h = cfg->h;
  P->h_rel = cfg->h_rel;
  P->rtol = cfg->rtol;
  P->atol = cfg->atol;
  P->h_cap_rel = cfg->h_cap_rel;
  P->max_steps = cfg->max_steps;
  P->lambda_max = cfg->lambda_max > 0.0 ? cfg->lambda_max : (double)INFINITY;  // <= 0 = no affine budget
  P->h_f = (float)cfg->h;
  P->h_rel_f = (float)cfg->h_rel;
  P->lambda_max_f = (float)P->lambda_max;
  if ((double)P->lambda_max_f < P->lambda_max) P->lambda_max_f = nextafterf(P->lambda_max_f, INFINITY);
  P->pad_f_ = 0.0f;
  P->r_cap = P->mc.r_horizon * (1.0 + cfg->eps_capture);
  P->r_esc = cfg->r_escape;
  P->ring_d = cfg->ring_half_angle;
  if (cfg->max_crossings > 0 || ring) {
    P->disk_r_in = (cfg->disk_r_in > 0.0) ? cfg->disk_r_in : isco_prograde(metric_id, P->mc);
    P->disk_r_out = cfg->disk_r_out;
    if (!(P->disk_r_out >= P->disk_r_in)) return GP_E_BAD_PARAM;
  }
  return GP_OK;
}

// ---- library-owned scratch for gp_trace_host -----------------------------------------------------
// One stream-ordered pool per device that keeps its memory between calls (release threshold = max): the
// default pool would hand 128 MiB back to the driver at every synchronisation and pay cudaMalloc again
// on the next call.  Created on first use under a mutex; allocations from it are per call.
int scratch_pool(cudaMemPool_t *out) {
  static cudaMemPool_t pools[64] = {};
  static std::mutex mu;
  int dev = 0;
  GP_CUDA(cudaGetDevice(&dev));
  if (dev < 0 || dev >= 64) return GP_E_UNSUPPORTED;
  std::lock_guard<std::mutex> lock(mu);
  if (!pools[dev]) {
    cudaMemPoolProps props = {};
    props.allocType = cudaMemAllocationTypePinned;
    props.location.type = cudaMemLocationTypeDevice;
    props.location.id = dev;
    cudaMemPool_t p = nullptr;
    GP_CUDA(cudaMemPoolCreate(&p, &props));
    unsigned long long keep = ~0ull;
    GP_CUDA(cudaMemPoolSetAttribute(p, cudaMemPoolAttrReleaseThreshold, &keep));
    pools[dev] = p;
  }
  *out = pools[dev];
  return GP_OK;
}

// ---- launch -----------------------------------------------------------------------------------
// Resident blocks per SM and the SM count are properties of (kernel, device): cached per device id
// under a mutex, so that a process may drive several devices and several host threads (the cache was
// bound to the first device in round 1).
constexpr int kMaxDevices = 64;
struct LaunchInfo {
  int n_sm;
  int per_sm;   // 0 = not computed yet
};
std::mutex g_launch_mutex;

template <class Kernel>
int launch_info(Kernel kernel, size_t smem, LaunchInfo *slot, LaunchInfo *out) {
  std::lock_guard<std::mutex> lock(g_launch_mutex);
  if (slot->per_sm == 0) {
    int dev = 0, n_sm = 0, occ = 0;
    GP_CUDA(cudaGetDevice(&dev));
    GP_CUDA(cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev));
    // dynamic shared memory beyond 48 KB (the disk variant of trace_dp54) needs the opt-in
    if (smem > 48 * 1024)
      GP_CUDA(cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    GP_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kernel, kBlock, smem));
    slot->n_sm = n_sm;
    slot->per_sm = occ < 1 ? 1 : occ;
  }
  *out = *slot;
  return GP_OK;
}

// OBJ: 0 no object, 1 thin disk with recorded crossings, 2 solid ring (scheme 2 only)
template <int METRIC, int OBJ>
int launch_one(const TraceParams &P, cudaStream_t stream) {
  static LaunchInfo cache[kMaxDevices][5];   // per device: dp54, rk4 FP64 / FP32 / mixed, dp54 mixed (zero-initialised)
  const bool dp54 = (P.scheme == 2);
  const int prec = P.precision;   // 0 FP64, 1 FP32, 2 FP32 equations + FP64 state
  // (the mixed adaptive kernels with an object are held to three blocks per SM by asking for the 60 KB their
  // park area used to need: measured on config 3 at rtol 1e-7, 29.1 ms with three blocks, 32.6 ms with four;
  // without an object four are faster for them too: 10.83 against 11.40 ms on the headline at rtol 1e-7)
  const size_t smem = dp54 ? ((prec == 2 && OBJ != 0) ? 16 * (size_t)kBlock * 30 : dp54_smem_bytes(OBJ != 0))
                           : (OBJ != 0 ? (prec == 1 ? sizeof(float) : sizeof(double)) * kBlock * kParkSlotsRk4 : 0) + kBirthQueueBytes;
  int dev = 0;
  GP_CUDA(cudaGetDevice(&dev));
  if (dev < 0 || dev >= kMaxDevices) return GP_E_UNSUPPORTED;
  LaunchInfo *slot = &cache[dev][dp54 ? (prec == 2 ? 4 : 0) : 1 + prec];
  LaunchInfo li;
  int rc;
  // persistent grid: every SM filled to its resident-block limit, never more lanes than rays
#define GP_GO(kernel_)                                                            \
  {                                                                               \
    rc = launch_info(kernel_, smem, slot, &li);                                   \
    if (rc) return rc;                                                            \
    long long want = ((long long)P.cc.ray_count + kBlock - 1) / kBlock;           \
    long long grid = (long long)li.n_sm * li.per_sm;                              \
    if (grid > want) grid = want;                                                 \
    if (grid < 1) grid = 1;                                                       \
    kernel_<<<(unsigned)grid, kBlock, smem, stream>>>(P);                         \
  }
  if (dp54) {
    if (prec == 2) {
      GP_GO((trace_dp54<METRIC, OBJ, float>))
    } else {
      GP_GO((trace_dp54<METRIC, OBJ>))
    }
  } else if (prec == 1) {
    GP_GO((trace_rk4<METRIC, OBJ, float>))
  } else if (prec == 2) {
    GP_GO((trace_rk4<METRIC, OBJ, float, double>))
  } else {
    GP_GO((trace_rk4<METRIC, OBJ, double>))
  }
#undef GP_GO
  GP_CUDA(cudaGetLastError());
  return GP_OK;
}

int launch_trace(int metric_id, const TraceParams &P, cudaStream_t stream) {
  const int obj = P.ring_d > 0.0 ? 2 : (P.max_crossings > 0 ? 1 : 0);
#define GP_LAUNCH(M_)                                              \
  (obj == 2 ? launch_one<M_, 2>(P, stream) : obj == 1 ? launch_one<M_, 1>(P, stream) : launch_one<M_, 0>(P, stream))
  switch (metric_id) {
    case GP_SCHWARZSCHILD: return GP_LAUNCH(METRIC_SCHW);
    case GP_KERR: return GP_LAUNCH(METRIC_KERR);
    default: return GP_LAUNCH(METRIC_MN);
  }
#undef GP_LAUNCH
}

// ---- step-level kernels (parity of rows a2-a5 in isolation) -------------------------------------
__global__ void k_init_conditions(const __grid_constant__ CameraConst cc, const __grid_constant__ MetricConst mc,
                                  double *states8, double *ab2) {
  long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= cc.ray_count) return;
  double alpha, beta, r, th, ph, pt, pr, pth, pph;
  alpha_beta(cc, cc.ray_begin + k * cc.ray_stride, alpha, beta);
  ray_birth(cc, mc, cc.ray_begin + k * cc.ray_stride, r, th, ph, pt, pr, pth, pph);
  double *s = states8 + 8 * k;
  s[0] = 0.0; s[1] = r; s[2] = th; s[3] = ph;
  s[4] = pt; s[5] = pr; s[6] = pth; s[7] = pph;
  if (ab2) {
    ab2[2 * k] = alpha;
    ab2[2 * k + 1] = beta;
  }
}

__global__ void k_eval_metric(int metric, const __grid_constant__ MetricConst mc, const double *rt2, long long n,
                              double *out15) {
  long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= n) return;
  double o[15];
  metric_inv15(metric, mc, rt2[2 * k], rt2[2 * k + 1], o);
  for (int i = 0; i < 15; ++i) out15[15 * k + i] = o[i];
}

template <int METRIC>
__global__ void k_eval_rhs(const __grid_constant__ MetricConst mc, const double *st8, long long n, double *rhs6) {
  long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= n) return;
  const double *s = st8 + 8 * k;
  Rhs o;
  rhs_eval<METRIC>(mc, s[4], s[7], s[1], s[2], s[5], s[6], o);
  double *d = rhs6 + 6 * k;
  d[0] = o.dt; d[1] = o.dr; d[2] = o.dth; d[3] = o.dph; d[4] = o.dpr; d[5] = o.dpth;
}

// FP64 FMA peak probe: 8 independent dependent chains per thread.
__global__ void __launch_bounds__(256) k_probe_fma(long long iters, double seed, double *sink) {
  double a0 = seed + threadIdx.x, a1 = a0 + 1.0, a2 = a0 + 2.0, a3 = a0 + 3.0, a4 = a0 + 4.0, a5 = a0 + 5.0,
         a6 = a0 + 6.0, a7 = a0 + 7.0;
  const double m = 0.999999, c = 1e-9;
  for (long long i = 0; i < iters; ++i) {
#pragma unroll
    for (int u = 0; u < 8; ++u) {
      a0 = fma(a0, m, c); a1 = fma(a1, m, c); a2 = fma(a2, m, c); a3 = fma(a3, m, c);
      a4 = fma(a4, m, c); a5 = fma(a5, m, c); a6 = fma(a6, m, c); a7 = fma(a7, m, c);
    }
  }
  double s = ((a0 + a1) + (a2 + a3)) + ((a4 + a5) + (a6 + a7));
  if (s == 123.456) *sink = s;  // keeps the chains alive without a store in practice
}

// ---- static scratch for gp_trace_static ----------------------------------------------------------
// Everything the trace kernels need besides the caller's inputs and outputs, in one file-scope array, so
// that gp_trace_static never allocates (gp.h): words 0-7 the counters block (word 0 = the atomic work
// counter), words 8-15 the two list counts of segmented tracing, then the two slot lists of
// GP_STATIC_MAX_RAYS entries each.  16 MiB + 128 bytes of .bss on every device that loads the library.
// In HOST code the name below is the host-side shadow of the symbol, not a device address: a kernel
// handed it would fault (or, where the GPU can reach host memory, scribble over the wrong memory).
// static_scratch() asks the runtime for the address, once per device, with that device current.
constexpr size_t kStaticHeadWords = 16;
static __device__ __align__(256) unsigned long long g_static_scratch[kStaticHeadWords + 2 * (size_t)GP_STATIC_MAX_RAYS];

int static_scratch(unsigned long long **out) {
  static unsigned long long *addr[kMaxDevices] = {};
  static std::mutex mu;
  int dev = 0;
  GP_CUDA(cudaGetDevice(&dev));
  if (dev < 0 || dev >= kMaxDevices) return GP_E_UNSUPPORTED;
  std::lock_guard<std::mutex> lock(mu);
  if (!addr[dev]) {
    void *p = nullptr;
    GP_CUDA(cudaGetSymbolAddress(&p, g_static_scratch));
    if (!p || ((uintptr_t)p & 255u) != 0) return GP_E_UNSUPPORTED;
    addr[dev] = (unsigned long long *)p;
  }
  *out = addr[dev];
  return GP_OK;
}

}  // namespace

// ---- exported entry points -----------------------------------------------------------------------
extern "C" {

int gp_trace(int metric_id, const gp_metric_params *metric, const gp_camera *camera,
             const gp_integrator_cfg *cfg, const gp_out_buffers *out, void *cuda_stream) {
  if (!out) return GP_E_NULL;
  TraceParams P;
  int rc = make_params(metric_id, metric, camera, cfg, &P);
  if (rc) return rc;
  const size_t n = (size_t)camera->ray_count;
  if (!out->counters) return GP_E_NULL;
  if (out->counters_bytes < 64) return GP_E_SIZE;
  if (((uintptr_t)out->counters & 7u) != 0) return GP_E_BAD_PARAM;
  if (n > 0) {
    if (!out->rays) return GP_E_NULL;
    if (out->rays_bytes < n * sizeof(gp_ray_record)) return GP_E_SIZE;
    if (((uintptr_t)out->rays & 31u) != 0) return GP_E_BAD_PARAM;
    if (cfg->max_crossings > 0 || cfg->ring_half_angle > 0.0) {
      if (!out->disk) return GP_E_NULL;
      if (out->disk_bytes < n * sizeof(gp_disk_record)) return GP_E_SIZE;
      if (((uintptr_t)out->disk & 7u) != 0) return GP_E_BAD_PARAM;
    }
  }
  P.rays = (gp_ray_record *)out->rays;
  P.disk = (gp_disk_record *)out->disk;
  P.counters = (unsigned long long *)out->counters;
  cudaStream_t stream = (cudaStream_t)cuda_stream;
  // Segmented tracing (gp.h, cfg.segment_steps): Manko-Novikov rays of the adaptive scheme that stall near
  // the singular horizon run to the step budget, 700 x a normal ray, and whichever lane draws them sets the
  // length of the launch.  Their state is parked after K attempted steps and the slots are redistributed over
  // all lanes by the next launch of the same kernel (round r + 1 reads the list round r wrote): the work
  // counter then balances steps, not rays.  Off unless asked for: measured on B200 it removes the end-of-image
  // tail (99 % of the rays done at 15.70 of 15.70 s instead of 14.60 of 15.78 s on config 4) but buys 0.5 % at
  // 2048^2 and 4 % at 1024^2 — the lanes that idle in the tail were not holding the others back.
  long long K = 0;
  if (metric_id == GP_MANKO_NOVIKOV && cfg->scheme == 2 && cfg->segment_steps != 0) {
    K = cfg->segment_steps > 0 ? cfg->segment_steps : (cfg->max_steps / 48 > 4096 ? cfg->max_steps / 48 : 4096);
    if (K >= cfg->max_steps) K = 0;   // one segment: nothing to park
  }
  if (K > 0 && (cfg->max_steps + K - 1) / K > 4096) return GP_E_BAD_PARAM;   // segment_steps too small for this budget
  GP_CUDA(cudaMemsetAsync(out->counters, 0, 64, stream));
  if (n == 0) return GP_OK;
  if (K == 0) return launch_trace(metric_id, P, stream);
  cudaMemPool_t pool = nullptr;
  rc = scratch_pool(&pool);
  if (rc) return rc;
  // scratch: two slot lists (n x 8 bytes each) and their two counts, stream-ordered, freed after the last round
  char *scratch = nullptr;
  const size_t list_b = (n * sizeof(long long) + 63) & ~(size_t)63;
  GP_CUDA(cudaMallocFromPoolAsync((void **)&scratch, 64 + 2 * list_b, pool, stream));
  unsigned long long *counts = (unsigned long long *)scratch;
  long long *lists[2] = {(long long *)(scratch + 64), (long long *)(scratch + 64 + list_b)};
  const long long rounds = (cfg->max_steps + K - 1) / K;
  P.seg_steps = K;
  cudaError_t e = cudaMemsetAsync(counts, 0, 64, stream);
  for (long long rd = 0; rd < rounds && e == cudaSuccess && rc == GP_OK; ++rd) {
    P.round = (int)rd;
    P.list_in = lists[rd & 1];
    P.list_in_count = counts + (rd & 1);
    P.list_out = lists[(rd + 1) & 1];
    P.list_out_count = counts + ((rd + 1) & 1);
    if (rd > 0) {
      e = cudaMemsetAsync(P.list_out_count, 0, sizeof(unsigned long long), stream);   // the list this round fills
      if (e == cudaSuccess) e = cudaMemsetAsync(out->counters, 0, sizeof(unsigned long long), stream);   // work counter
    }
    if (e == cudaSuccess) rc = launch_trace(metric_id, P, stream);
  }
  cudaError_t e2 = cudaFreeAsync(scratch, stream);
  if (rc != GP_OK) return rc;
  if (e != cudaSuccess) return cuda_fail(e);
  if (e2 != cudaSuccess) return cuda_fail(e2);
  return GP_OK;
}

int gp_trace_host(int metric_id, const gp_metric_params *metric, const gp_camera *camera,
                  const gp_integrator_cfg *cfg, const gp_out_buffers *out, void *cuda_stream) {
  if (!out || !camera || !cfg) return GP_E_NULL;
  TraceParams P;
  int rc = make_params(metric_id, metric, camera, cfg, &P);
  if (rc) return rc;
  const size_t n = (size_t)camera->ray_count;
  const bool disk = cfg->max_crossings > 0 || cfg->ring_half_angle > 0.0;
  const size_t rays_b = n * sizeof(gp_ray_record), disk_b = disk ? n * sizeof(gp_disk_record) : 0;
  if (n > 0) {
    if (!out->rays) return GP_E_NULL;
    if (out->rays_bytes < rays_b) return GP_E_SIZE;
    if (disk && !out->disk) return GP_E_NULL;
    if (disk && out->disk_bytes < disk_b) return GP_E_SIZE;
  }
  if (out->counters && out->counters_bytes < 64) return GP_E_SIZE;
  cudaStream_t stream = (cudaStream_t)cuda_stream;
  cudaMemPool_t pool = nullptr;
  rc = scratch_pool(&pool);
  if (rc) return rc;
  // Pinned (page-locked, mapped) host buffers are written by the kernel itself: a lane stores its
  // 128-byte record once, when its ray ends, so the records cross PCIe while the other rays are still
  // being integrated and no device-to-host copy remains after the kernel.  Pageable buffers take the
  // staged path below (device scratch + cudaMemcpyAsync).
  cudaPointerAttributes ar, ad;
  bool direct = n > 0 && cudaPointerGetAttributes(&ar, out->rays) == cudaSuccess &&
                ar.type == cudaMemoryTypeHost && ar.devicePointer != nullptr;
  if (direct && disk)
    direct = cudaPointerGetAttributes(&ad, out->disk) == cudaSuccess && ad.type == cudaMemoryTypeHost &&
             ad.devicePointer != nullptr;
  cudaGetLastError();  // a pageable pointer leaves cudaErrorInvalidValue behind on old drivers
  // one scratch allocation per call, stream-ordered: counters | ray records | disk records (the last two
  // only on the staged path).  Nothing is shared between calls, so concurrent calls on different streams
  // and host threads are independent.
  const size_t off_rays = 64, off_disk = off_rays + ((rays_b + 63) & ~(size_t)63);
  const size_t scratch_b = direct ? 64 : off_disk + disk_b + 64;
  char *scratch = nullptr;
  GP_CUDA(cudaMallocFromPoolAsync((void **)&scratch, scratch_b, pool, stream));
  gp_out_buffers dev;
  dev.counters = scratch;
  dev.counters_bytes = 64;
  dev.rays = direct ? ar.devicePointer : (void *)(scratch + off_rays);
  dev.rays_bytes = rays_b;
  dev.disk = disk ? (direct ? ad.devicePointer : (void *)(scratch + off_disk)) : nullptr;
  dev.disk_bytes = disk_b;
  rc = gp_trace(metric_id, metric, camera, cfg, &dev, cuda_stream);
  cudaError_t e = cudaSuccess;
  if (rc == GP_OK) {
    if (!direct && n > 0) e = cudaMemcpyAsync(out->rays, dev.rays, rays_b, cudaMemcpyDeviceToHost, stream);
    if (!direct && e == cudaSuccess && disk && n > 0)
      e = cudaMemcpyAsync(out->disk, dev.disk, disk_b, cudaMemcpyDeviceToHost, stream);
    if (e == cudaSuccess && out->counters)
      e = cudaMemcpyAsync(out->counters, dev.counters, 64, cudaMemcpyDeviceToHost, stream);
  }
  cudaError_t e2 = cudaFreeAsync(scratch, stream);
  cudaError_t e3 = cudaStreamSynchronize(stream);
  if (rc != GP_OK) return rc;
  if (e != cudaSuccess) return cuda_fail(e);
  if (e2 != cudaSuccess) return cuda_fail(e2);
  if (e3 != cudaSuccess) return cuda_fail(e3);
  return GP_OK;
}

int gp_trace_static(int metric_id, const gp_metric_params *metric, const gp_camera *camera,
                    const gp_integrator_cfg *cfg, const gp_out_buffers *out, void *cuda_stream) {
  if (!out) return GP_E_NULL;
  TraceParams P;
  int rc = make_params(metric_id, metric, camera, cfg, &P);
  if (rc) return rc;
  const size_t n = (size_t)camera->ray_count;
  if (n > (size_t)GP_STATIC_MAX_RAYS) return GP_E_STATIC_LIMIT;
  if (out->counters) {
    if (out->counters_bytes < 64) return GP_E_SIZE;
    if (((uintptr_t)out->counters & 7u) != 0) return GP_E_BAD_PARAM;
  }
  if (n > 0) {
    if (!out->rays) return GP_E_NULL;
    if (out->rays_bytes < n * sizeof(gp_ray_record)) return GP_E_SIZE;
    if (((uintptr_t)out->rays & 31u) != 0) return GP_E_BAD_PARAM;
    if (cfg->max_crossings > 0 || cfg->ring_half_angle > 0.0) {
      if (!out->disk) return GP_E_NULL;
      if (out->disk_bytes < n * sizeof(gp_disk_record)) return GP_E_SIZE;
      if (((uintptr_t)out->disk & 7u) != 0) return GP_E_BAD_PARAM;
    }
  }
  // segment length: the rule of gp_trace
  long long K = 0;
  if (metric_id == GP_MANKO_NOVIKOV && cfg->scheme == 2 && cfg->segment_steps != 0) {
    K = cfg->segment_steps > 0 ? cfg->segment_steps : (cfg->max_steps / 48 > 4096 ? cfg->max_steps / 48 : 4096);
    if (K >= cfg->max_steps) K = 0;
  }
  if (K > 0 && (cfg->max_steps + K - 1) / K > 4096) return GP_E_BAD_PARAM;
  unsigned long long *S = nullptr;   // DEVICE address of g_static_scratch on the current device
  rc = static_scratch(&S);
  if (rc) return rc;
  cudaStream_t stream = (cudaStream_t)cuda_stream;
  P.rays = (gp_ray_record *)out->rays;
  P.disk = (gp_disk_record *)out->disk;
  P.counters = S;
  // the array keeps the last call's totals and list counts: clear the 128 bytes that must start at zero
  GP_CUDA(cudaMemsetAsync(S, 0, kStaticHeadWords * sizeof(unsigned long long), stream));
  cudaError_t e = cudaSuccess;
  if (n > 0 && K == 0) {
    rc = launch_trace(metric_id, P, stream);
  } else if (n > 0) {
    unsigned long long *counts = S + 8;
    long long *lists[2] = {(long long *)(S + kStaticHeadWords),
                           (long long *)(S + kStaticHeadWords + (size_t)GP_STATIC_MAX_RAYS)};
    const long long rounds = (cfg->max_steps + K - 1) / K;
    P.seg_steps = K;
    for (long long rd = 0; rd < rounds && e == cudaSuccess && rc == GP_OK; ++rd) {
      P.round = (int)rd;
      P.list_in = lists[rd & 1];
      P.list_in_count = counts + (rd & 1);
      P.list_out = lists[(rd + 1) & 1];
      P.list_out_count = counts + ((rd + 1) & 1);
      if (rd > 0) {
        e = cudaMemsetAsync(P.list_out_count, 0, sizeof(unsigned long long), stream);
        if (e == cudaSuccess) e = cudaMemsetAsync(S, 0, sizeof(unsigned long long), stream);   // work counter
      }
      if (e == cudaSuccess) rc = launch_trace(metric_id, P, stream);
    }
  }
  if (rc != GP_OK) return rc;
  if (e != cudaSuccess) return cuda_fail(e);
  if (out->counters) GP_CUDA(cudaMemcpyAsync(out->counters, S, 64, cudaMemcpyDeviceToDevice, stream));
  return GP_OK;
}

int gp_init_conditions(int metric_id, const gp_metric_params *metric, const gp_camera *camera, void *states8,
                       size_t states_bytes, void *alpha_beta2, size_t ab_bytes, void *cuda_stream) {
  if (!metric || !camera) return GP_E_NULL;
  MetricConst mc;
  int rc = make_metric(metric_id, metric, &mc);
  if (rc) return rc;
  CameraConst cc;
  rc = make_camera(metric_id, mc, camera, 0.0, &cc);
  if (rc) return rc;
  const size_t n = (size_t)camera->ray_count;
  if (n == 0) return GP_OK;
  if (!states8) return GP_E_NULL;
  if (states_bytes < n * 64) return GP_E_SIZE;
  if (alpha_beta2 && ab_bytes < n * 16) return GP_E_SIZE;
  if (((uintptr_t)states8 & 7u) != 0 || ((uintptr_t)alpha_beta2 & 7u) != 0) return GP_E_BAD_PARAM;
  const unsigned grid = (unsigned)((n + 255) / 256);
  k_init_conditions<<<grid, 256, 0, (cudaStream_t)cuda_stream>>>(cc, mc, (double *)states8, (double *)alpha_beta2);
  GP_CUDA(cudaGetLastError());
  return GP_OK;
}

int gp_eval_metric(int metric_id, const gp_metric_params *metric, const void *r_theta2, int64_t n, void *out15,
                   size_t out_bytes, void *cuda_stream) {
  if (!metric) return GP_E_NULL;
  MetricConst mc;
  int rc = make_metric(metric_id, metric, &mc);
  if (rc) return rc;
  if (n < 0) return GP_E_BAD_PARAM;
  if (n == 0) return GP_OK;
  if (!r_theta2 || !out15) return GP_E_NULL;
  if (out_bytes < (size_t)n * 15 * sizeof(double)) return GP_E_SIZE;
  if (((uintptr_t)r_theta2 & 7u) != 0 || ((uintptr_t)out15 & 7u) != 0) return GP_E_BAD_PARAM;
  const unsigned grid = (unsigned)((n + 127) / 128);
  k_eval_metric<<<grid, 128, 0, (cudaStream_t)cuda_stream>>>(metric_id, mc, (const double *)r_theta2, n,
                                                             (double *)out15);
  GP_CUDA(cudaGetLastError());
  return GP_OK;
}

int gp_eval_rhs(int metric_id, const gp_metric_params *metric, const void *states8, int64_t n, void *rhs6,
                size_t rhs_bytes, void *cuda_stream) {
  if (!metric) return GP_E_NULL;
  MetricConst mc;
  int rc = make_metric(metric_id, metric, &mc);
  if (rc) return rc;
  if (n < 0) return GP_E_BAD_PARAM;
  if (n == 0) return GP_OK;
  if (!states8 || !rhs6) return GP_E_NULL;
  if (rhs_bytes < (size_t)n * 6 * sizeof(double)) return GP_E_SIZE;
  if (((uintptr_t)states8 & 7u) != 0 || ((uintptr_t)rhs6 & 7u) != 0) return GP_E_BAD_PARAM;
  const unsigned grid = (unsigned)((n + 127) / 128);
  cudaStream_t st = (cudaStream_t)cuda_stream;
  if (metric_id == GP_SCHWARZSCHILD)
    k_eval_rhs<METRIC_SCHW><<<grid, 128, 0, st>>>(mc, (const double *)states8, n, (double *)rhs6);
  else if (metric_id == GP_KERR)
    k_eval_rhs<METRIC_KERR><<<grid, 128, 0, st>>>(mc, (const double *)states8, n, (double *)rhs6);
  else
    k_eval_rhs<METRIC_MN><<<grid, 128, 0, st>>>(mc, (const double *)states8, n, (double *)rhs6);
  GP_CUDA(cudaGetLastError());
  return GP_OK;
}

int gp_probe_fp64_fma(int64_t iters, void *scratch, size_t scratch_bytes, double *flops_out, void *cuda_stream) {
  if (!scratch || !flops_out) return GP_E_NULL;
  if (scratch_bytes < 8) return GP_E_SIZE;
  if (iters <= 0) return GP_E_BAD_PARAM;
  int dev = 0, n_sm = 0;
  GP_CUDA(cudaGetDevice(&dev));
  GP_CUDA(cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev));
  const int blocks = n_sm * 8, threads = 256;  // 2048 resident threads per SM
  k_probe_fma<<<blocks, threads, 0, (cudaStream_t)cuda_stream>>>(iters, 0.5, (double *)scratch);
  GP_CUDA(cudaGetLastError());
  *flops_out = 2.0 * 64.0 * (double)iters * (double)blocks * (double)threads;
  return GP_OK;
}

int gp_integrate_orbits(int metric_id, const gp_metric_params *metric, const gp_orbit_cfg *cfg,
                        const void *states8, int64_t n, void *samples, size_t samples_bytes, void *status,
                        size_t status_bytes, void *n_steps, size_t n_steps_bytes, void *cuda_stream) {
  if (!metric || !cfg) return GP_E_NULL;
  OrbitParams P;
  memset(&P, 0, sizeof(P));
  int rc = make_metric(metric_id, metric, &P.mc);
  if (rc) return rc;
  if (!(cfg->rtol > 0.0) || !(cfg->atol >= 0.0) || !(cfg->h0 > 0.0) || !(cfg->h_max > 0.0) ||
      !(cfg->lambda_end > 0.0) || !(cfg->eps_capture >= 0.0) || cfg->n_samples < 1 || cfg->max_steps < 0 || n < 0)
    return GP_E_BAD_PARAM;
  if (!isfinite(cfg->rtol) || !isfinite(cfg->atol) || !isfinite(cfg->h0) || !isfinite(cfg->h_max) ||
      !isfinite(cfg->lambda_end) || !isfinite(cfg->eps_capture))
    return GP_E_BAD_PARAM;
  if (n == 0) return GP_OK;
  if (!states8 || !samples || !status || !n_steps) return GP_E_NULL;
  if (samples_bytes < (size_t)n * (size_t)cfg->n_samples * 64 || status_bytes < (size_t)n * 4 ||
      n_steps_bytes < (size_t)n * 8)
    return GP_E_SIZE;
  // samples are written with 256-bit stores, states read as doubles, status / n_steps as 32 / 64-bit words
  if (((uintptr_t)samples & 31u) != 0 || ((uintptr_t)states8 & 7u) != 0 || ((uintptr_t)status & 3u) != 0 ||
      ((uintptr_t)n_steps & 7u) != 0)
    return GP_E_BAD_PARAM;
  P.rtol = cfg->rtol; P.atol = cfg->atol; P.h0 = cfg->h0; P.h_max = cfg->h_max; P.lambda_end = cfg->lambda_end;
  P.r_cap = P.mc.r_horizon * (1.0 + cfg->eps_capture);
  P.n = n; P.n_samples = cfg->n_samples; P.max_steps = cfg->max_steps;
  P.states8 = (const double *)states8;
  P.samples = (double *)samples;
  P.status = (unsigned *)status;
  P.n_steps = (unsigned long long *)n_steps;
  const unsigned grid = (unsigned)((n + 127) / 128);
  cudaStream_t st = (cudaStream_t)cuda_stream;
  if (metric_id == GP_SCHWARZSCHILD) k_integrate_orbits<METRIC_SCHW><<<grid, 128, 0, st>>>(P);
  else if (metric_id == GP_KERR) k_integrate_orbits<METRIC_KERR><<<grid, 128, 0, st>>>(P);
  else k_integrate_orbits<METRIC_MN><<<grid, 128, 0, st>>>(P);
  GP_CUDA(cudaGetLastError());
  return GP_OK;
}

int gp_shade(const gp_shade_cfg *cfg, const void *rays, size_t rays_bytes, const void *disk, size_t disk_bytes,
             void *rgba8, size_t rgba_bytes, void *cuda_stream) {
  if (!cfg || !rays || !rgba8) return GP_E_NULL;
  if (cfg->width <= 0 || cfg->height <= 0 || cfg->supersample <= 0 || cfg->supersample > 16) return GP_E_BAD_PARAM;
  if (cfg->mode < 0 || cfg->mode > 2) return GP_E_BAD_PARAM;
  if (cfg->mode == 0 && !(cfg->grid_step_deg > 0.0 && cfg->grid_half_width_deg >= 0.0 &&
                          isfinite(cfg->grid_step_deg) && isfinite(cfg->grid_half_width_deg)))
    return GP_E_BAD_PARAM;
  if (cfg->mode == 1 && (cfg->tex_width <= 0 || cfg->tex_height <= 0 || cfg->tex_width > (1 << 30) ||
                         cfg->tex_height > (1 << 30)))
    return GP_E_BAD_PARAM;
  if (cfg->mode == 2 && !(cfg->time_period > 0.0 && isfinite(cfg->time_period))) return GP_E_BAD_PARAM;
  if (cfg->disk_overlay != 0 && cfg->disk_overlay != 1) return GP_E_BAD_PARAM;
  if (cfg->disk_overlay) {
    if (!disk) return GP_E_NULL;
    if (!(cfg->g_lo < 1.0) || !(cfg->g_hi > 1.0) || !isfinite(cfg->g_lo) || !isfinite(cfg->g_hi)) return GP_E_BAD_PARAM;
  }
  const long long S = cfg->supersample;
  const size_t n = (size_t)cfg->width * (size_t)cfg->height * (size_t)(S * S);
  const size_t npix = (size_t)cfg->width * (size_t)cfg->height;
  if (rays_bytes < n * sizeof(gp_ray_record)) return GP_E_SIZE;
  if (cfg->disk_overlay && disk_bytes < n * sizeof(gp_disk_record)) return GP_E_SIZE;
  if (rgba_bytes < npix * 4) return GP_E_SIZE;
  // records are read with 128-bit loads, disk records as doubles, pixels written as 32-bit words
  if (((uintptr_t)rays & 15u) != 0 || ((uintptr_t)rgba8 & 3u) != 0 || (cfg->disk_overlay && ((uintptr_t)disk & 7u) != 0))
    return GP_E_BAD_PARAM;
  ShadeParams P;
  memset(&P, 0, sizeof(P));
  P.W = cfg->width; P.H = cfg->height; P.S = S;
  P.mode = cfg->mode; P.disk_overlay = cfg->disk_overlay;
  const double pi = 3.14159265358979323846;
  P.step_rad = cfg->grid_step_deg * (pi / 180.0);
  P.hw_rad = cfg->grid_half_width_deg * (pi / 180.0);
  P.tw = cfg->tex_width; P.th = cfg->tex_height; P.tex_seed = cfg->tex_seed;
  P.time_period = cfg->time_period; P.g_lo = cfg->g_lo; P.g_hi = cfg->g_hi;
  P.rays = (const gp_ray_record *)rays;
  P.disk = (const gp_disk_record *)disk;
  P.rgba = (unsigned char *)rgba8;
  const unsigned grid = (unsigned)((npix + 255) / 256);
  k_shade<<<grid, 256, 0, (cudaStream_t)cuda_stream>>>(P);
  GP_CUDA(cudaGetLastError());
  return GP_OK;
}

int gp_metric_radii(int metric_id, const gp_metric_params *metric, double *r_horizon, double *r_isco) {
  if (!metric || !r_horizon || !r_isco) return GP_E_NULL;
  MetricConst mc;
  int rc = make_metric(metric_id, metric, &mc);
  if (rc) return rc;
  *r_horizon = mc.r_horizon;
  *r_isco = isco_prograde(metric_id, mc);
  return GP_OK;
}

size_t gp_ray_record_size(void) { return sizeof(gp_ray_record); }
size_t gp_disk_record_size(void) { return sizeof(gp_disk_record); }
size_t gp_counters_size(void) { return 64; }
int64_t gp_static_max_rays(void) { return GP_STATIC_MAX_RAYS; }
int gp_version(void) { return GP_VERSION; }

const char *gp_strerror(int code) {
  static thread_local char buf[320];
  switch (code) {
    case GP_OK: return "ok";
    case GP_E_BAD_METRIC: return "unknown metric id";
    case GP_E_BAD_PARAM: return "parameter out of range";
    case GP_E_NULL: return "null pointer";
    case GP_E_SIZE: return "buffer too small";
    case GP_E_UNSUPPORTED: return "variant not built";
    case GP_E_STATIC_LIMIT:
      return "gp_trace_static: ray_count exceeds GP_STATIC_MAX_RAYS (1048576), the capacity of the library's "
             "static scratch; tile the image with ray_begin / ray_count or call gp_trace";
    case GP_E_CUDA:
      snprintf(buf, sizeof(buf), "CUDA error: %s", g_cuda_msg);
      return buf;
  }
  return "unknown error code";
}

}  // extern "C"
