// C ABI of the B200-native RA-MPPI hot path (see include/ra_mppi.h).
// Host side: context, validation, kernel dispatch, CUDA-graph closed loop.
#include "../../include/ra_mppi.h"

#include <cuda_runtime.h>

#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include "launchers.h"
#include "rollout.cuh"
#include "update.cuh"

using namespace ra;

struct ra_mppi_ctx {
  ra_mppi_config cfg{};
  Params p{};
  int rc = 1;          // realisations interleaved per lane in the rollout kernel
  bool half = false;   // M <= 16: half a warp per sample (2 rc samples per warp)
  int noise_variant = 0;
  int n_sm = 0;        // multiprocessors of cfg.device (grid sizing of the small kernels)
  RolloutLaunchFn rollout = nullptr;
  // device allocations owned by the context
  float4* d_circles = nullptr;
  float4* d_costmap = nullptr;  // quad-texel table: allocation
  float4* d_quadmap = nullptr;  // ... and the table inside it, placed so that it does not straddle a 4 GiB boundary
  float2* d_u_raw = nullptr;
  float4* d_ce = nullptr;
  double* d_S = nullptr;
  float* d_cvar = nullptr;
  double* d_pen = nullptr;
  double* d_split = nullptr;   // [kMaxUpdateSplits][2+2T] partials of the update's sample ranges
  unsigned int* d_done = nullptr;   // ticket counter of the update kernel's CTAs (its last CTA combines and re-arms it)
  float* d_w_mat = nullptr;
  LoopState* d_loop = nullptr;
  // closed-loop graph cache
  // host-buffer staging (ra_mppi_step_host) and optional kernel timing
  // ra_mppi_step_host: staging buffer [8 + 2T] floats = { iteration (u64), x0 (6 floats), v [T,2] } on the device and, pinned,
  // on the host (one copy each way whatever memory the caller passes), and the whole call captured once as a CUDA graph
  // (H2D copy, the step's kernels reading the iteration from the staging buffer, D2H copy): one launch call per step
  float* d_stage = nullptr;
  float* h_stage = nullptr;
  cudaGraphExec_t host_graph = nullptr;
  bool host_graph_failed = false;
  bool pdl = true;     // programmatic dependent launch of the kernels that follow a kernel on the caller's stream
  bool timing = false;
  bool timed = false;  // ev_k0 / ev_k1 hold a rollout-kernel interval recorded outside a stream capture
  cudaEvent_t ev_k0 = nullptr, ev_k1 = nullptr;
  // the nominal rollout (A2) runs beside the noisy rollouts (A3-A7) on this stream, forked from and
  // joined back into the caller's stream with the two events (captured as parallel graph branches)
  cudaStream_t side = nullptr;
  cudaEvent_t ev_fork = nullptr, ev_join = nullptr;
  cudaGraphExec_t graph_exec = nullptr;
  float *g_x0 = nullptr, *g_v = nullptr, *g_log = nullptr;
  std::string err;
};

namespace {

constexpr int kMaxUpdateSplits = 64;

ra_status fail(ra_mppi_ctx* c, ra_status s, const std::string& msg) {
  if (c) c->err = msg;
  return s;
}

ra_status cuda_fail(ra_mppi_ctx* c, cudaError_t e, const char* what) {
  if (e == cudaSuccess) return RA_OK;
  const ra_status s = (e == cudaErrorMemoryAllocation) ? RA_ENOMEM : RA_ECUDA;
  return fail(c, s, std::string(what) + ": " + cudaGetErrorString(e));
}

#define RA_CUDA(ctx, call)                                  \
  do {                                                      \
    cudaError_t e__ = (call);                               \
    if (e__ != cudaSuccess) return cuda_fail(ctx, e__, #call); \
  } while (0)

bool finite_nonneg(float x) { return std::isfinite(x) && x >= 0.0f; }

// alpha and eta arrive as fp32: the decimal the caller meant lies within one fp32 ulp of a value below 1,
// i.e. within 2^-23 of the number received, so (1 - x) n is known to 2^-23 n.  The guard against that
// representation error is therefore 2^-23 n (0.7f -> (1-alpha) 10 = 3.0000001 must count 3); the fp64 oracle
// uses 1e-9.  The two sides agree unless the true (1 - x) n lies within 2^-23 n above an integer.
constexpr double kFp32Ulp = 1.1920928955078125e-07;   // 2^-23

// k_tail = ceil((1-alpha) M) (G11), clamped to [1, M].
int tail_count(double alpha, int M) {
  int k = (int)std::ceil((1.0 - alpha) * (double)M - kFp32Ulp * (double)M);
  return k < 1 ? 1 : (k > M ? M : k);
}

// K0 = ceil((1-eta) K): samples with global index below K0 carry the mean control (Alg.1 l.7-10).
int mean_count(double eta, int K_total) {
  int k = (int)std::ceil((1.0 - eta) * (double)K_total - kFp32Ulp * (double)K_total);
  return k < 0 ? 0 : (k > K_total ? K_total : k);
}

// Makes cfg.device current for the duration of an entry point and restores the caller's device afterwards.
struct DeviceGuard {
  int prev = -1;
  bool ok = true;
  explicit DeviceGuard(int device) {
    if (cudaGetDevice(&prev) != cudaSuccess) { prev = -1; ok = false; return; }
    if (prev != device) ok = cudaSetDevice(device) == cudaSuccess; else prev = -1;
  }
  ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
  DeviceGuard(const DeviceGuard&) = delete;
  DeviceGuard& operator=(const DeviceGuard&) = delete;
};
#define RA_ON_DEVICE(ctx)                                                      \
  DeviceGuard device_guard__((ctx)->cfg.device);                               \
  if (!device_guard__.ok) return fail((ctx), RA_ECUDA, "cudaSetDevice failed")

const char* validate(const ra_mppi_config* cfg, const ra_mppi_env* env, ra_status* st) {
  *st = RA_EINVAL;
  if (cfg->struct_size != sizeof(ra_mppi_config)) return "struct_size mismatch";
  if (cfg->K <= 0 || cfg->M <= 0 || cfg->T <= 0) return "K, M, T must be positive";
  if (cfg->K_total == 0 && cfg->k_offset != 0) return "k_offset needs K_total";
  if (cfg->K_total != 0 && (cfg->k_offset < 0 || cfg->K_total < cfg->K || cfg->k_offset > cfg->K_total - cfg->K))
    return "shard [k_offset, k_offset + K) must lie inside [0, K_total)";
  if (!(cfg->dt > 0.0f) || !std::isfinite(cfg->dt)) return "dt must be positive";
  if (cfg->dyn != RA_DYN_KINEMATIC_BICYCLE && cfg->dyn != RA_DYN_SINGLE_TRACK) return "unknown dyn";
  if (cfg->nominal < RA_NOM_GOAL || cfg->nominal > RA_NOM_RACING) return "unknown nominal cost";
  if (cfg->risk < RA_RISK_CIRCLES || cfg->risk > RA_RISK_NOMINAL) return "unknown risk cost";
  if (cfg->noise_kind < RA_NOISE_GAUSSIAN || cfg->noise_kind > RA_NOISE_JUMP) return "unknown noise kind";
  if (cfg->noise_mode != RA_NOISE_FUSED && cfg->noise_mode != RA_NOISE_MATERIALISED) return "unknown noise mode";
  if (!(cfg->alpha > 0.0f && cfg->alpha < 1.0f)) return "alpha must be in (0,1) (PAPER.md:87)";
  if (!(cfg->lambda > 0.0f) || !std::isfinite(cfg->lambda)) return "lambda must be positive";
  if (!finite_nonneg(cfg->gamma)) return "gamma must be >= 0";
  if (!(cfg->eta >= 0.0f && cfg->eta < 1.0f)) return "eta must be in [0,1)";
  if (!(cfg->B > 0.0f) || !std::isfinite(cfg->B)) return "B must be positive";
  if (!std::isfinite(cfg->A) || !std::isfinite(cfg->C_u)) return "A, C_u must be finite";
  for (int i = 0; i < 2; ++i) {
    if (!finite_nonneg(cfg->sigma_eps[i])) return "sigma_eps must be >= 0";
    if (!(cfg->u_min[i] <= cfg->u_max[i])) return "u_min must be <= u_max";
  }
  for (int i = 0; i < 6; ++i)
    if (!finite_nonneg(cfg->sigma_w[i])) return "sigma_w must be >= 0";
  if (cfg->dyn == RA_DYN_KINEMATIC_BICYCLE && !(cfg->dyn_p[0] > 0.0f)) return "wheelbase must be positive";
  if (cfg->dyn == RA_DYN_SINGLE_TRACK && (!(cfg->dyn_p[0] > 0.0f) || !(cfg->dyn_p[1] > 0.0f) || !(cfg->dyn_p[6] > 0.0f)))
    return "single-track needs m, Iz, vx_floor > 0";
  if (cfg->nominal == RA_NOM_ELLIPSE_TRACK && (!(cfg->nom_p[0] > 0.0f) || !(cfg->nom_p[1] > 0.0f)))
    return "track semi-axes must be positive";
  const bool uses_circles = cfg->risk == RA_RISK_CIRCLES || cfg->nominal == RA_NOM_RACING;
  if (uses_circles) {
    if (!env || env->n_circles < 0 || (env->n_circles > 0 && !env->circles)) return "circle costs need env->circles";
  }
  if (cfg->nominal == RA_NOM_RACING && (!(cfg->nom_p[0] > 0.0f) || !(cfg->nom_p[1] > 0.0f) || !(cfg->nom_p[2] > 0.0f)))
    return "racing track needs ax, ay, rc > 0";
  if (cfg->risk == RA_RISK_COSTMAP) {
    if (!env || !env->costmap || env->map_h < 1 || env->map_w < 1 || !(env->map_res > 0.0f))
      return "costmap risk needs env->costmap";
    if (env->map_h > (1 << 20) || env->map_w > (1 << 20)) return "costmap side above 2^20 cells";
    if ((long long)(env->map_h + 1) * (env->map_w + 1) >= (1LL << 28)) return "costmap table above 4 GB";
  }
  if (cfg->risk == RA_RISK_LINEAR_STATE) {
    const int nx = cfg->dyn == RA_DYN_SINGLE_TRACK ? 6 : 4;
    if (!(cfg->risk_p[1] >= 0.0f && cfg->risk_p[1] < (float)nx)) return "linear risk index out of range";
  }
  if (cfg->noise_kind == RA_NOISE_JUMP && !(cfg->noise_p[0] >= 0.0f && cfg->noise_p[0] <= 1.0f))
    return "jump probability must be in [0,1]";
  if (cfg->risk == RA_RISK_CIRCLES && (!finite_nonneg(cfg->risk_p[1]) || !std::isfinite(cfg->risk_p[0])))
    return "circle risk needs a finite weight and a finite margin >= 0";
  *st = RA_EUNSUPPORTED;
  if (cfg->M > RA_MAX_M) return "M above RA_MAX_M";
  if (cfg->T > RA_MAX_T) return "T above RA_MAX_T";
  if (uses_circles && env->n_circles > kMaxCirclesSmem) return "too many circles";
  if (cfg->risk == RA_RISK_NOMINAL && cfg->nominal != RA_NOM_RACING) return "l = q is built for the racing costs only";
  *st = RA_OK;
  return nullptr;
}

RolloutLaunchFn pick_rollout(int dyn, int risk) {
  static const RolloutLaunchFn table[2][4] = {
      {launch_rollout_0_0, launch_rollout_0_1, launch_rollout_0_2, launch_rollout_0_3},
      {launch_rollout_1_0, launch_rollout_1_1, launch_rollout_1_2, launch_rollout_1_3}};
  return table[dyn][risk];
}

void philox_round_keys(uint64_t seed, uint32_t rk[20]) {
  uint32_t k0 = (uint32_t)(seed & 0xFFFFFFFFull), k1 = (uint32_t)(seed >> 32);
  for (int r = 0; r < 10; ++r) {
    rk[2 * r] = k0; rk[2 * r + 1] = k1;
    k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
  }
}

template <typename T>
cudaError_t dev_alloc(T** p, size_t n) { return cudaMalloc(reinterpret_cast<void**>(p), n * sizeof(T)); }

// Copies the environment into the context (synchronously).  first = allocate: the obstacle buffer holds
// kMaxCirclesSmem records and the costmap table its create-time size, so later uploads never allocate.
ra_status upload_env(ra_mppi_ctx* c, const ra_mppi_env* env, bool first) {
  const ra_mppi_config* cfg = &c->cfg;
  Params& p = c->p;
  if (cfg->risk == RA_RISK_CIRCLES || cfg->nominal == RA_NOM_RACING) {
    // (cx, cy, r + margin, r): the hinge risk cost (BASELINE configs) tests against r + margin, the indicator cost (22)
    // of the racing nominal cost against the bare radius r (it has no margin), also when both are in use
    const float margin = cfg->risk == RA_RISK_CIRCLES ? cfg->risk_p[1] : 0.0f;
    std::vector<float4> h((size_t)std::max(env->n_circles, 1));
    for (int i = 0; i < env->n_circles; ++i)
      h[i] = make_float4(env->circles[3 * i], env->circles[3 * i + 1], env->circles[3 * i + 2] + margin,
                         env->circles[3 * i + 2]);
    if (first && dev_alloc(&c->d_circles, (size_t)kMaxCirclesSmem) != cudaSuccess) return fail(c, RA_ENOMEM, "alloc circles");
    if (cuda_fail(c, cudaMemcpy(c->d_circles, h.data(), h.size() * sizeof(float4), cudaMemcpyHostToDevice), "copy circles"))
      return RA_ECUDA;
    p.n_circles = env->n_circles;
    p.circles = c->d_circles;
  }
  if (cfg->risk == RA_RISK_COSTMAP) {
    // risk-weighted bilinear coefficient table (models.cuh) around grid corner (jx-1/2, jy-1/2)
    const int H = env->map_h, Wd = env->map_w;
    const size_t n = (size_t)(H + 1) * (Wd + 1);
    std::vector<float4> q(n);
    auto at = [&](int iy, int ix) {
      iy = iy < 0 ? 0 : (iy > H - 1 ? H - 1 : iy);
      ix = ix < 0 ? 0 : (ix > Wd - 1 ? Wd - 1 : ix);
      return (double)env->costmap[(size_t)iy * Wd + ix];
    };
    const double w = (double)cfg->risk_p[0];
    for (int jy = 0; jy <= H; ++jy)
      for (int jx = 0; jx <= Wd; ++jx) {
        const double c00 = at(jy - 1, jx - 1), c01 = at(jy - 1, jx), c10 = at(jy, jx - 1), c11 = at(jy, jx);
        q[(size_t)jy * (Wd + 1) + jx] = make_float4((float)(w * c00), (float)(w * (c01 - c00)), (float)(w * (c10 - c00)),
                                                    (float)(w * (c11 - c10 - c01 + c00)));
      }
    if (first) {
      // The kernel forms a lookup address as (high word of the table) : (low word + 16 idx) with one 32-bit add, so the
      // table must lie inside one 4 GiB-aligned window (its size is < 4 GiB, validated).  An allocation that straddles a
      // boundary (about one in a thousand for a 4 MB table) is replaced by one of twice the size, which always holds an
      // aligned copy.
      const size_t bytes = n * sizeof(float4);
      auto straddles = [bytes](const void* q0) { return ((reinterpret_cast<uintptr_t>(q0) & 0xFFFFFFFFull) + bytes) > (1ull << 32); };
      if (dev_alloc(&c->d_costmap, n) != cudaSuccess) return fail(c, RA_ENOMEM, "alloc costmap");
      c->d_quadmap = c->d_costmap;
      if (straddles(c->d_costmap)) {
        cudaFree(c->d_costmap); c->d_costmap = nullptr;
        if (dev_alloc(&c->d_costmap, 2 * n) != cudaSuccess) return fail(c, RA_ENOMEM, "alloc costmap");
        c->d_quadmap = c->d_costmap;
        if (straddles(c->d_costmap))   // start the table at the boundary inside the allocation
          c->d_quadmap = reinterpret_cast<float4*>((reinterpret_cast<uintptr_t>(c->d_costmap) + bytes) & ~0xFFFFFFFFull);
      }
    }
    if (cuda_fail(c, cudaMemcpy(c->d_quadmap, q.data(), n * sizeof(float4), cudaMemcpyHostToDevice), "copy costmap"))
      return RA_ECUDA;
    p.quadmap = c->d_quadmap;
    p.map_h = env->map_h; p.map_w = env->map_w;
    p.map_inv_res = (float)(1.0 / (double)env->map_res);
    p.map_ox = env->map_ox; p.map_oy = env->map_oy;
  }
  return RA_OK;
}

}  // namespace

// Why the calling thread's last ra_mppi_create failed: there is no context yet to hold the text (ra_mppi_create_error).
namespace {
thread_local char g_create_error[256] = "";
ra_status create_fail(ra_status st, const char* fmt, int a = 0, int b = 0) {
  std::snprintf(g_create_error, sizeof g_create_error, fmt, a, b);
  return st;
}
}  // namespace

extern "C" {

const char* ra_mppi_create_error(void) { return g_create_error; }

ra_status ra_mppi_create(const ra_mppi_config* cfg, const ra_mppi_env* env, ra_mppi_ctx** out) {
  g_create_error[0] = '\0';
  if (!out) return create_fail(RA_EINVAL, "null output pointer");
  *out = nullptr;
  if (!cfg) return create_fail(RA_EINVAL, "null config");
  ra_status st;
  if (const char* why = validate(cfg, env, &st)) {
    std::snprintf(g_create_error, sizeof g_create_error, "%s", why);
    return st;
  }
  int n_dev = 0;
  if (cudaGetDeviceCount(&n_dev) != cudaSuccess || cfg->device < 0 || cfg->device >= n_dev)
    return create_fail(RA_ECUDA, "no CUDA device %d (this library has no CPU fallback)", cfg->device);
  cudaDeviceProp prop{};
  if (cudaGetDeviceProperties(&prop, cfg->device) != cudaSuccess) return create_fail(RA_ECUDA, "cudaGetDeviceProperties failed");
  if (prop.major != 10) return create_fail(RA_EUNSUPPORTED, "device is sm_%d%d, built for sm_100a only", prop.major, prop.minor);
  ra_mppi_ctx* c = new (std::nothrow) ra_mppi_ctx();
  if (!c) return create_fail(RA_ENOMEM, "out of host memory");
  c->cfg = *cfg;
  // the context's own error text (set by upload_env and the CUDA wrappers) outlives it in the thread's create-error slot
  auto bail = [&](ra_status s, const char* what = "") {
    std::snprintf(g_create_error, sizeof g_create_error, "%s%s%s", what, (what[0] && !c->err.empty()) ? ": " : "", c->err.c_str());
    ra_mppi_destroy(c);
    return s;
  };
  DeviceGuard on_device(cfg->device);   // the caller's current device is restored on return
  if (!on_device.ok) return bail(RA_ECUDA, "cudaSetDevice failed");
  c->n_sm = prop.multiProcessorCount;

  Params& p = c->p;
  p.K = cfg->K; p.M = cfg->M; p.T = cfg->T;
  const int K_total = cfg->K_total ? cfg->K_total : cfg->K;
  p.k_off = cfg->k_offset;
  p.K0 = mean_count((double)cfg->eta, K_total);   // on the global index
  p.device = cfg->device;
  p.k_tail = tail_count((double)cfg->alpha, cfg->M);
  c->half = cfg->M <= 16;
  p.G = c->half ? 16 : 32;
  p.R_total = (cfg->M + p.G - 1) / p.G;
  // Work split of the rollout kernel (measured on B200, profiles/r1c): a warp interleaves RC slots
  // of 32 realisations per lane (RC = 4 when the slot count divides by 4, else 2), and the
  // ceil(R_total / RC) groups of one control sample go to as many warps (wps, a power of two <= 8),
  // so every warp runs one group: shorter CTAs fill the SMs at small K (the paper's 1024 x 300
  // workload: 5 groups -> 8 warps) and cut the wave tail at large K.
  p.wps = 1;
  // M <= 16: a warp carries 2 rc samples.  Two slots per lane halve the per-state-step share of the obstacle culling, but
  // also the number of warps: measured on B200 (profiles/r2), rc = 2 wins from K = 65536 (0.308 -> 0.281 ms) and loses below
  // K = 16384 (0.093 -> 0.098 ms; K = 1024: 0.034 -> 0.045 ms), where the GPU is not full.
  c->rc = (c->half && cfg->K >= 32768) ? 2 : 1;
  if (!c->half) {
    c->rc = (p.R_total >= 4 && p.R_total % 4 == 0) ? 4 : (p.R_total >= 2 ? 2 : 1);
    // The costmap kernel prefers two slots per lane at 80 registers and 3 CTAs/SM (6 warps per scheduler instead of 4) now
    // that it is co-limited by issue slots and the MUFU queue: C3 rollout 0.359 -> 0.343 ms.  The circle and single-track
    // kernels keep four (their per-step culling and their dynamics amortise over the slots: RC = 2 costs them 4-6 %).
    // The materialised-noise variant streams four rows per step and lane better (5.1 against 4.5 TB/s).
    if (cfg->risk == RA_RISK_COSTMAP && cfg->dyn == RA_DYN_KINEMATIC_BICYCLE && cfg->noise_mode == RA_NOISE_FUSED && c->rc == 4) c->rc = 2;
    const int groups = (p.R_total + c->rc - 1) / c->rc;
    while (p.wps < 8 && p.wps < groups) p.wps *= 2;
  }
  {
    // shared-memory carveout (percent of the 228 KB unified L1) that holds three rollout CTAs; the nominal-rollout
    // kernel asks for the same split so both kernels can share an SM
    const bool circ = cfg->risk == RA_RISK_CIRCLES || cfg->nominal == RA_NOM_RACING;
    const size_t ce_slots = c->half ? 2 * c->rc * kRolloutWarps : kRolloutWarps / p.wps;
    const size_t smem_cta = (circ && env ? (size_t)((env->n_circles + 31) & ~31) * sizeof(float4) : 0) +
                            ce_slots * cfg->T * sizeof(float4) +
                            (size_t)kRolloutWarps * (c->half ? c->rc : p.R_total) * 32 * sizeof(uint32_t);
    const size_t need = 3 * (smem_cta + 1024);
    p.carveout = need <= 57 * 1024 ? 25 : (need <= 114 * 1024 ? 50 : 100);
  }
  p.nx = cfg->dyn == RA_DYN_SINGLE_TRACK ? 6 : 4;
  p.dyn = cfg->dyn; p.noise_kind = cfg->noise_kind;
  p.dt = cfg->dt;
  std::memcpy(p.dyn_p, cfg->dyn_p, sizeof p.dyn_p);
  if (cfg->dyn == RA_DYN_SINGLE_TRACK) {
    p.dyn_q[0] = (float)(1.0 / (double)cfg->dyn_p[0]);
    p.dyn_q[1] = (float)(1.0 / (double)cfg->dyn_p[1]);
  } else {
    p.dyn_q[0] = (float)((double)cfg->dt / (double)cfg->dyn_p[0]);   // dt / L of the yaw update
  }
  std::memcpy(p.nom_p, cfg->nom_p, sizeof p.nom_p);
  if (cfg->nominal == RA_NOM_ELLIPSE_TRACK) {
    p.nom_q[0] = (float)(1.0 / (double)cfg->nom_p[0]);
    p.nom_q[1] = (float)(1.0 / (double)cfg->nom_p[1]);
  }
  std::memcpy(p.risk_p, cfg->risk_p, sizeof p.risk_p);
  std::memcpy(p.noise_p, cfg->noise_p, sizeof p.noise_p);
  std::memcpy(p.sigma_w, cfg->sigma_w, sizeof p.sigma_w);
  {
    // rng.cuh: Gaussian a = sqrt(-log2 u1)(cos, sin)(2 pi (u2 - 1/2)) = -z / sqrt(2 ln 2); uniform a = z;
    // jump a = -(unit direction)
    const double c = cfg->noise_kind == RA_NOISE_GAUSSIAN ? -std::sqrt(2.0 * std::log(2.0))
                     : (cfg->noise_kind == RA_NOISE_JUMP ? -1.0 : 1.0);
    for (int i = 0; i < 6; ++i) p.wscale[i] = (float)(c * (double)cfg->sigma_w[i]);
  }
  for (int i = 0; i < 2; ++i) {
    p.u_min[i] = cfg->u_min[i]; p.u_max[i] = cfg->u_max[i];
    p.sigma_eps[i] = cfg->sigma_eps[i];
    // gamma v^T Sigma^-1 u (3) PAPER.md:47; a component with sigma_eps = 0 is not sampled and is skipped
    p.ctrl_w[i] = cfg->sigma_eps[i] > 0.0f
                      ? (float)((double)cfg->gamma / ((double)cfg->sigma_eps[i] * (double)cfg->sigma_eps[i]))
                      : 0.0f;
  }
  p.neg_log2e_over_lambda = (float)(-1.4426950408889634 / (double)cfg->lambda);
  p.A = cfg->A; p.B = cfg->B; p.C_u = cfg->C_u;
  philox_round_keys(cfg->seed, p.rk);
  c->noise_variant = cfg->noise_mode == RA_NOISE_MATERIALISED ? NOISE_MATERIALISED : cfg->noise_kind;
  c->rollout = pick_rollout(cfg->dyn, cfg->risk);

  // environment copies (buffers sized once; ra_mppi_set_env refills them)
  if (ra_status st_env = upload_env(c, env, true)) return bail(st_env, "environment");
  // scratch
  const size_t KT = (size_t)cfg->K * cfg->T;
  if (dev_alloc(&c->d_u_raw, KT) != cudaSuccess || dev_alloc(&c->d_ce, KT) != cudaSuccess ||
      dev_alloc(&c->d_S, (size_t)cfg->K) != cudaSuccess || dev_alloc(&c->d_cvar, (size_t)cfg->K) != cudaSuccess ||
      dev_alloc(&c->d_pen, (size_t)cfg->K) != cudaSuccess || dev_alloc(&c->d_split, (size_t)kMaxUpdateSplits * (2 + 2 * cfg->T)) != cudaSuccess || dev_alloc(&c->d_loop, 1) != cudaSuccess ||
      dev_alloc(&c->d_done, 1) != cudaSuccess ||
      dev_alloc(&c->d_stage, (size_t)(8 + 2 * cfg->T)) != cudaSuccess ||
      cudaHostAlloc(reinterpret_cast<void**>(&c->h_stage), (size_t)(8 + 2 * cfg->T) * sizeof(float), cudaHostAllocDefault) != cudaSuccess)
    return bail(RA_ENOMEM, "device or pinned-host allocation of the context scratch failed");
  p.u_raw = c->d_u_raw; p.ce = c->d_ce; p.S = c->d_S; p.cvar = c->d_cvar; p.pen = c->d_pen;
  if (cudaMemset(c->d_loop, 0, sizeof(LoopState)) != cudaSuccess || cudaMemset(c->d_done, 0, sizeof(unsigned int)) != cudaSuccess ||
      cudaMemset(c->d_cvar, 0, (size_t)cfg->K * sizeof(float)) != cudaSuccess ||
      cudaMemset(c->d_pen, 0, (size_t)cfg->K * sizeof(double)) != cudaSuccess)   // A = 0 steps never write them
    return bail(RA_ECUDA, "cudaMemset of the context scratch failed");
  if (cudaStreamCreateWithFlags(&c->side, cudaStreamNonBlocking) != cudaSuccess ||
      cudaEventCreateWithFlags(&c->ev_fork, cudaEventDisableTiming) != cudaSuccess ||
      cudaEventCreateWithFlags(&c->ev_join, cudaEventDisableTiming) != cudaSuccess)
    return bail(RA_ECUDA, "side stream / event creation failed");
  p.M_pad = p.R_total * p.G;
  if (cfg->noise_mode == RA_NOISE_MATERIALISED) {
    const size_t n = KT * (size_t)p.nx * (size_t)p.M_pad;
    if (dev_alloc(&c->d_w_mat, n) != cudaSuccess) return bail(RA_ENOMEM, "device allocation of the materialised noise tensor failed");
    p.w_mat = c->d_w_mat;
  }
  p.d_iter = nullptr; p.iter_imm = 0;
  *out = c;
  return RA_OK;
}

ra_status ra_mppi_destroy(ra_mppi_ctx* c) {
  if (!c) return RA_OK;
  DeviceGuard on_device(c->cfg.device);
  if (c->graph_exec) cudaGraphExecDestroy(c->graph_exec);
  if (c->host_graph) cudaGraphExecDestroy(c->host_graph);
  cudaFree(c->d_circles); cudaFree(c->d_costmap); cudaFree(c->d_u_raw); cudaFree(c->d_ce);
  cudaFree(c->d_stage);
  if (c->h_stage) cudaFreeHost(c->h_stage);
  if (c->ev_fork) cudaEventDestroy(c->ev_fork);
  if (c->ev_join) cudaEventDestroy(c->ev_join);
  if (c->side) cudaStreamDestroy(c->side);
  if (c->ev_k0) cudaEventDestroy(c->ev_k0);
  if (c->ev_k1) cudaEventDestroy(c->ev_k1);
  cudaFree(c->d_S); cudaFree(c->d_cvar); cudaFree(c->d_pen); cudaFree(c->d_split); cudaFree(c->d_w_mat); cudaFree(c->d_loop); cudaFree(c->d_done);
  delete c;
  return RA_OK;
}

ra_status ra_mppi_set_env(ra_mppi_ctx* c, const ra_mppi_env* env) {
  if (!c) return RA_EINVAL;
  const ra_mppi_config* cfg = &c->cfg;
  const bool uses_circles = cfg->risk == RA_RISK_CIRCLES || cfg->nominal == RA_NOM_RACING;
  if (!env) return fail(c, RA_EINVAL, "null env");
  if (uses_circles && (env->n_circles < 0 || (env->n_circles > 0 && !env->circles)))
    return fail(c, RA_EINVAL, "circle costs need env->circles");
  if (uses_circles && env->n_circles > kMaxCirclesSmem) return fail(c, RA_EUNSUPPORTED, "too many circles");
  if (cfg->risk == RA_RISK_COSTMAP &&
      (!env->costmap || env->map_h != c->p.map_h || env->map_w != c->p.map_w || !(env->map_res > 0.0f)))
    return fail(c, RA_EINVAL, "costmap must keep the size it had at ra_mppi_create");
  RA_ON_DEVICE(c);
  // earlier launches may still read the old copies; a captured graph holds the old sizes in its kernel arguments
  RA_CUDA(c, cudaDeviceSynchronize());
  if (c->graph_exec) { cudaGraphExecDestroy(c->graph_exec); c->graph_exec = nullptr; }
  if (c->host_graph) { cudaGraphExecDestroy(c->host_graph); c->host_graph = nullptr; }
  return upload_env(c, env, false);
}

const char* ra_mppi_last_error(const ra_mppi_ctx* c) { return c ? c->err.c_str() : "null context"; }

ra_status ra_mppi_query_counts(const ra_mppi_config* cfg, int32_t* h_k_tail, int32_t* h_K0) {
  if (!cfg || cfg->struct_size != sizeof(ra_mppi_config) || cfg->M <= 0 || cfg->K <= 0) return RA_EINVAL;
  if (!(cfg->alpha > 0.0f && cfg->alpha < 1.0f) || !(cfg->eta >= 0.0f && cfg->eta < 1.0f)) return RA_EINVAL;
  if (h_k_tail) *h_k_tail = tail_count((double)cfg->alpha, cfg->M);
  if (h_K0) *h_K0 = mean_count((double)cfg->eta, cfg->K_total ? cfg->K_total : cfg->K);
  return RA_OK;
}


}  // extern "C"

namespace {

cudaError_t launch_sample(const ra_mppi_ctx* c, const Params& p, const float* d_v, cudaStream_t s) {
  const dim3 grid((p.K + kSampleKB - 1) / kSampleKB, (p.T * kSampleKB + kSampleThreads - 1) / kSampleThreads);
  if (c->cfg.dyn == 0) sample_kernel<0><<<grid, kSampleThreads, 0, s>>>(p, d_v);
  else sample_kernel<1><<<grid, kSampleThreads, 0, s>>>(p, d_v);
  return cudaGetLastError();   // a plain launch: the first kernel of a step depends on everything before it
}

cudaError_t launch_nominal(const ra_mppi_ctx* c, const Params& p, const float* d_x0, const float* d_v,
                           cudaStream_t s, bool pdl) {
  const int grid = (p.K + kNominalThreads - 1) / kNominalThreads;
  const int dyn = c->cfg.dyn, nom = c->cfg.nominal;
#define RA_NOMK(D, N)                                                                                          \
  do {                                                                                                         \
    static std::atomic<int> carveout_set[kMaxDevices];   /* same L1 / shared-memory split as the rollout kernel */ \
    if (const cudaError_t e = set_func_attr_once(carveout_set, p.device, nominal_kernel<D, N>,                  \
                                                 cudaFuncAttributePreferredSharedMemoryCarveout, p.carveout))  \
      return e;                                                                                                \
    return launch_kernel(nominal_kernel<D, N>, dim3(grid), dim3(kNominalThreads), 0, s, pdl, p, d_x0, d_v);    \
  } while (0)
  if (dyn == 0) { if (nom == 0) RA_NOMK(0, 0); else if (nom == 1) RA_NOMK(0, 1); else RA_NOMK(0, 2); }
  else { if (nom == 0) RA_NOMK(1, 0); else if (nom == 1) RA_NOMK(1, 1); else RA_NOMK(1, 2); }
#undef RA_NOMK
}

template <int NX>
cudaError_t launch_materialise(const ra_mppi_ctx* c, const Params& p, cudaStream_t s) {
  const long long n = (long long)p.K * p.T * p.M_pad;
  const int grid = (int)std::min<long long>((n + 255) / 256, (long long)c->n_sm * 16);
  switch (c->cfg.noise_kind) {
    case RA_NOISE_GAUSSIAN: materialise_noise_kernel<NX, NOISE_GAUSSIAN><<<grid, 256, 0, s>>>(p, c->d_w_mat); break;
    case RA_NOISE_UNIFORM: materialise_noise_kernel<NX, NOISE_UNIFORM><<<grid, 256, 0, s>>>(p, c->d_w_mat); break;
    default: materialise_noise_kernel<NX, NOISE_JUMP><<<grid, 256, 0, s>>>(p, c->d_w_mat); break;
  }
  return cudaGetLastError();
}

// Alg.1 l.3-29: sampling, nominal and noisy rollouts, CVaR, soft filter -> context scratch.
ra_status enqueue_costs(ra_mppi_ctx* c, const Params& p, const float* d_x0, const float* d_v, float* d_L,
                        float* d_xT, cudaStream_t s, bool diagnostics) {
  // A = 0 is the baseline MPPI of section II: S~ = S by (14)-(16), so unless the caller
  // asks for the risk diagnostics the M noisy rollouts are not needed at all.
  if (c->cfg.A == 0.0f && !diagnostics) {
    // pen stays zero on this path: zeroed at create, and again after every diagnostics pass of an A = 0 context (below);
    // the update reads S + pen only, so a stale cvar from such a pass is harmless
    RA_CUDA(c, launch_sample(c, p, d_v, s));
    RA_CUDA(c, launch_nominal(c, p, d_x0, d_v, s, c->pdl));
    return RA_OK;
  }
  if (c->cfg.noise_mode == RA_NOISE_MATERIALISED)
    RA_CUDA(c, p.nx == 4 ? launch_materialise<4>(c, p, s) : launch_materialise<6>(c, p, s));
  RA_CUDA(c, launch_sample(c, p, d_v, s));
  // fork: the K*T nominal rollout needs only the sampled controls and hides under the K*M*T noisy ones
  RA_CUDA(c, cudaEventRecord(c->ev_fork, s));
  RA_CUDA(c, cudaStreamWaitEvent(c->side, c->ev_fork, 0));
  RA_CUDA(c, launch_nominal(c, p, d_x0, d_v, c->side, false));
  RA_CUDA(c, cudaEventRecord(c->ev_join, c->side));
  // the timing pair is recorded on live streams only: an event recorded during capture has no elapsed time
  cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
  if (c->timing) RA_CUDA(c, cudaStreamIsCapturing(s, &cap));
  const bool time_it = c->timing && cap == cudaStreamCaptureStatusNone;
  if (time_it) RA_CUDA(c, cudaEventRecord(c->ev_k0, s));
  // A plain launch, on purpose: as a programmatic dependent of the sampling kernel the rollout CTAs become resident
  // before the nominal kernel on the side stream is released, fill every SM (2 CTAs x 256 threads x 128 registers) and
  // push the nominal rollout behind the whole first wave -- measured on B200: C1 step 0.051 -> 0.068 ms, closed loop
  // p50 0.152 -> 0.162 ms (profiles/r2).  The weights/update kernel behind it is the programmatic dependent.
  RA_CUDA(c, c->rollout(p, c->noise_variant, c->rc, c->half, d_x0, d_L, d_xT, s, false));
  if (time_it) { RA_CUDA(c, cudaEventRecord(c->ev_k1, s)); c->timed = true; }
  RA_CUDA(c, cudaStreamWaitEvent(s, c->ev_join, 0));   // join
  // A = 0 with diagnostics: the kernel wrote pen = A * cvar, which is NaN for a diverged rollout (0 * inf) and would then
  // sit in S~ of every later A = 0 step, which skips the noisy rollouts and never rewrites it.  J_C is 0 by (14) at A = 0.
  if (c->cfg.A == 0.0f) RA_CUDA(c, cudaMemsetAsync(c->d_pen, 0, sizeof(double) * (size_t)p.K, s));
  return RA_OK;
}

// Alg.1 l.31: weights (17) and update (4) from the context scratch.  One CTA per (horizon step, sample range); a range
// is what one CTA caches in registers (kUpdateCached samples per thread), so the kernel is a single wave of small CTAs
// whose ranges are combined like the shards of the K-sharded step.
int update_splits(const ra_mppi_ctx* c) {
  const int per_cta = kUpdateThreads * kUpdateCached;
  return std::max(1, std::min(kMaxUpdateSplits, (c->p.K + per_cta - 1) / per_cta));
}

// steps of the horizon one update CTA takes: as many as keep the grid at about two CTAs per SM (at least one)
int update_steps_per_cta(const ra_mppi_ctx* c, int splits) {
  const int want = (c->p.T * splits) / (2 * std::max(c->n_sm, 1));
  return std::max(1, std::min(kUpdateMaxSteps, want));
}

ra_status enqueue_update(ra_mppi_ctx* c, const Params& p, float* d_v_out, cudaStream_t s, UpdateTail tail) {
  // a programmatic dependent of the rollout kernel (of the nominal kernel when A = 0); the join with the side stream
  // before it is a full dependency.  A timed step keeps plain launches.
  const int splits = update_splits(c), steps = update_steps_per_cta(c, splits);
  RA_CUDA(c, launch_kernel(weights_update_kernel<double>, dim3((p.T + steps - 1) / steps, splits), dim3(kUpdateThreads), 0, s,
                           c->pdl && !c->timing, p, (const double*)p.S, (const double*)p.pen, (const float2*)p.u_raw, 1LL,
                           (long long)p.K, d_v_out, (float*)nullptr, (float*)nullptr, c->d_split, c->d_done, tail, steps));
  return RA_OK;
}

// The shard's share of (17)/(4) for the K-sharded step.
ra_status enqueue_partial(ra_mppi_ctx* c, const Params& p, double* d_partial, cudaStream_t s) {
  RA_CUDA(c, launch_kernel(weights_update_kernel<double>, dim3(p.T, 1), dim3(kUpdateThreads), 0, s, c->pdl && !c->timing, p,
                           (const double*)p.S, (const double*)p.pen, (const float2*)p.u_raw, 1LL, (long long)p.K,
                           (float*)nullptr, (float*)nullptr, (float*)nullptr, d_partial, (unsigned int*)nullptr,
                           UpdateTail{nullptr, nullptr, nullptr}, 1));
  return RA_OK;
}

cudaError_t launch_plant(const Params& p, float* d_x0, float* d_v, float* d_u, float* d_log, LoopState* loop,
                         cudaStream_t s) {
  plant_shift_kernel<<<1, 128, 0, s>>>(p, d_x0, d_v, d_u, d_log, loop);
  return cudaGetLastError();
}

Params with_iteration(const ra_mppi_ctx* c, uint64_t iteration) {
  Params p = c->p;
  p.d_iter = nullptr;
  p.iter_imm = iteration;
  return p;
}

}  // namespace

extern "C" {

ra_status ra_mppi_rollout_variant(const ra_mppi_ctx* c, int32_t* h_variant) {
  if (!c || !h_variant) return RA_EINVAL;
  h_variant[0] = c->cfg.dyn; h_variant[1] = c->cfg.risk; h_variant[2] = c->noise_variant;
  h_variant[3] = c->rc; h_variant[4] = c->half ? 1 : 0;
  return RA_OK;
}

ra_status ra_mppi_step(ra_mppi_ctx* c, const float* d_x0, float* d_v, uint64_t iteration, void* stream) {
  if (!c) return RA_EINVAL;
  if (!d_x0 || !d_v) return fail(c, RA_EINVAL, "null device pointer");
  RA_ON_DEVICE(c);
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  const Params p = with_iteration(c, iteration);
  if (ra_status st = enqueue_costs(c, p, d_x0, d_v, nullptr, nullptr, s, false)) return st;
  return enqueue_update(c, p, d_v, s, UpdateTail{nullptr, nullptr, nullptr});
}

ra_status ra_mppi_step_partial(ra_mppi_ctx* c, const float* d_x0, const float* d_v, uint64_t iteration,
                               double* d_partial, void* stream) {
  if (!c) return RA_EINVAL;
  if (!d_x0 || !d_v || !d_partial) return fail(c, RA_EINVAL, "null device pointer");
  RA_ON_DEVICE(c);
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  const Params p = with_iteration(c, iteration);
  if (ra_status st = enqueue_costs(c, p, d_x0, d_v, nullptr, nullptr, s, false)) return st;
  return enqueue_partial(c, p, d_partial, s);
}

ra_status ra_mppi_combine_partials(ra_mppi_ctx* c, const double* d_partials, int32_t n_parts, float* d_v_plus,
                                   void* stream) {
  if (!c) return RA_EINVAL;
  if (!d_partials || !d_v_plus || n_parts < 1) return fail(c, RA_EINVAL, "bad arguments");
  RA_ON_DEVICE(c);
  combine_partials_kernel<<<1, 256, 0, static_cast<cudaStream_t>(stream)>>>(c->p, d_partials, n_parts, d_v_plus);
  RA_CUDA(c, cudaGetLastError());
  return RA_OK;
}

ra_status ra_mppi_rollout_costs(ra_mppi_ctx* c, const float* d_x0, const float* d_v, uint64_t iteration,
                                float* d_S, float* d_cvar, float* d_S_tilde, float* d_L, float* d_xT,
                                float* d_u, void* stream) {
  if (!c) return RA_EINVAL;
  if (!d_x0 || !d_v) return fail(c, RA_EINVAL, "null device pointer");
  RA_ON_DEVICE(c);
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  const Params p = with_iteration(c, iteration);
  if (ra_status st = enqueue_costs(c, p, d_x0, d_v, d_L, d_xT, s, true)) return st;
  if (d_S || d_cvar || d_S_tilde) {
    export_costs_kernel<<<(p.K + 255) / 256, 256, 0, s>>>(p, d_S, d_cvar, d_S_tilde);
    RA_CUDA(c, cudaGetLastError());
  }
  if (d_u) {
    export_u_kernel<<<c->n_sm * 4, 256, 0, s>>>(p, reinterpret_cast<float2*>(d_u));
    RA_CUDA(c, cudaGetLastError());
  }
  return RA_OK;
}

ra_status ra_mppi_weights_update(ra_mppi_ctx* c, const float* d_S_tilde, const float* d_u, float* d_v_plus,
                                 float* d_w, float* d_stats, void* stream) {
  if (!c) return RA_EINVAL;
  if (!d_S_tilde || !d_u || !d_v_plus) return fail(c, RA_EINVAL, "null device pointer");
  RA_ON_DEVICE(c);
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  const Params p = with_iteration(c, 0);
  weights_update_kernel<float><<<p.T, kUpdateThreads, 0, s>>>(
      p, d_S_tilde, nullptr, reinterpret_cast<const float2*>(d_u), (long long)p.T, 1LL, d_v_plus, d_w, d_stats, nullptr,
      nullptr, UpdateTail{nullptr, nullptr, nullptr}, 1);
  RA_CUDA(c, cudaGetLastError());
  return RA_OK;
}

ra_status ra_mppi_plant_shift(ra_mppi_ctx* c, float* d_x0, float* d_v, float* d_u_applied, uint64_t iteration,
                              void* stream) {
  if (!c) return RA_EINVAL;
  if (!d_x0 || !d_v) return fail(c, RA_EINVAL, "null device pointer");
  RA_ON_DEVICE(c);
  const Params p = with_iteration(c, iteration);
  RA_CUDA(c, launch_plant(p, d_x0, d_v, d_u_applied, nullptr, nullptr, static_cast<cudaStream_t>(stream)));
  return RA_OK;
}

ra_status ra_mppi_step_host(ra_mppi_ctx* c, const float* h_x0, float* h_v, uint64_t iteration, void* stream) {
  if (!c) return RA_EINVAL;
  if (!h_x0 || !h_v) return fail(c, RA_EINVAL, "null host pointer");
  RA_ON_DEVICE(c);
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  float* d_x0 = c->d_stage + 2;
  float* d_v = c->d_stage + 8;
  const size_t nv = (size_t)2 * c->p.T;
  std::memcpy(c->h_stage, &iteration, sizeof(uint64_t));
  std::memcpy(c->h_stage + 2, h_x0, (size_t)c->p.nx * sizeof(float));
  std::memcpy(c->h_stage + 8, h_v, nv * sizeof(float));
  // The whole call as one graph launch (captured on first use; a timed step and a failed capture take the call-by-call path)
  if (!c->host_graph && !c->host_graph_failed && !c->timing) {
    cudaStream_t cs = nullptr;
    cudaGraph_t graph = nullptr;
    ra_status st = RA_OK;
    if (cudaStreamCreateWithFlags(&cs, cudaStreamNonBlocking) == cudaSuccess &&
        cudaStreamBeginCapture(cs, cudaStreamCaptureModeThreadLocal) == cudaSuccess) {
      Params p = c->p;
      p.d_iter = reinterpret_cast<const unsigned long long*>(c->d_stage);
      p.iter_imm = 0;
      if (cudaMemcpyAsync(c->d_stage, c->h_stage, (8 + nv) * sizeof(float), cudaMemcpyHostToDevice, cs) != cudaSuccess) st = RA_ECUDA;
      if (st == RA_OK) st = enqueue_costs(c, p, d_x0, d_v, nullptr, nullptr, cs, false);
      if (st == RA_OK) st = enqueue_update(c, p, d_v, cs, UpdateTail{nullptr, nullptr, nullptr});
      if (st == RA_OK && cudaMemcpyAsync(c->h_stage + 8, d_v, nv * sizeof(float), cudaMemcpyDeviceToHost, cs) != cudaSuccess) st = RA_ECUDA;
      const cudaError_t e = cudaStreamEndCapture(cs, &graph);
      if (st != RA_OK || e != cudaSuccess || cudaGraphInstantiate(&c->host_graph, graph, 0) != cudaSuccess) c->host_graph = nullptr;
      if (graph) cudaGraphDestroy(graph);
    }
    if (cs) cudaStreamDestroy(cs);
    if (!c->host_graph) { c->host_graph_failed = true; (void)cudaGetLastError(); }
  }
  if (c->host_graph && !c->timing) {
    RA_CUDA(c, cudaGraphLaunch(c->host_graph, s));
  } else {
    RA_CUDA(c, cudaMemcpyAsync(c->d_stage, c->h_stage, (8 + nv) * sizeof(float), cudaMemcpyHostToDevice, s));
    if (ra_status st = ra_mppi_step(c, d_x0, d_v, iteration, stream)) return st;
    RA_CUDA(c, cudaMemcpyAsync(c->h_stage + 8, d_v, nv * sizeof(float), cudaMemcpyDeviceToHost, s));
  }
  RA_CUDA(c, cudaStreamSynchronize(s));
  std::memcpy(h_v, c->h_stage + 8, nv * sizeof(float));
  return RA_OK;
}

ra_status ra_mppi_enable_kernel_timing(ra_mppi_ctx* c, int32_t enable) {
  if (!c) return RA_EINVAL;
  RA_ON_DEVICE(c);
  if (enable && !c->ev_k0) {
    RA_CUDA(c, cudaEventCreate(&c->ev_k0));
    RA_CUDA(c, cudaEventCreate(&c->ev_k1));
  }
  c->timing = enable != 0;
  return RA_OK;
}

ra_status ra_mppi_last_rollout_ms(ra_mppi_ctx* c, float* h_ms) {
  if (!c) return RA_EINVAL;
  if (!h_ms || !c->ev_k0) return fail(c, RA_EINVAL, "kernel timing was never enabled");
  if (!c->timed)
    return fail(c, RA_EINVAL, "no rollout kernel has been timed: A = 0 steps launch none, and steps captured into a CUDA "
                              "graph record no timing events");
  RA_ON_DEVICE(c);
  RA_CUDA(c, cudaEventSynchronize(c->ev_k1));
  RA_CUDA(c, cudaEventElapsedTime(h_ms, c->ev_k0, c->ev_k1));
  return RA_OK;
}

ra_status ra_mppi_export_costs_f64(ra_mppi_ctx* c, double* d_S64, double* d_S_tilde64, void* stream) {
  if (!c) return RA_EINVAL;
  RA_ON_DEVICE(c);
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  if (d_S64 || d_S_tilde64) {
    export_costs_f64_kernel<<<(c->p.K + 255) / 256, 256, 0, s>>>(c->p, d_S64, d_S_tilde64);
    RA_CUDA(c, cudaGetLastError());
  }
  return RA_OK;
}

int32_t ra_mppi_launches_per_step(const ra_mppi_ctx* c) {
  if (!c) return 0;
  if (c->cfg.A == 0.0f) return 3;   // baseline MPPI: sampling, nominal rollout, weights/update
  return 4 + (c->cfg.noise_mode == RA_NOISE_MATERIALISED ? 1 : 0);   // + noisy rollouts (+ noise generator)
}

ra_status ra_mppi_philox(ra_mppi_ctx* c, const uint32_t* d_ctr, int32_t n, uint32_t* d_out, void* stream) {
  if (!c) return RA_EINVAL;
  if (!d_ctr || !d_out || n < 0) return fail(c, RA_EINVAL, "bad arguments");
  if (n == 0) return RA_OK;
  RA_ON_DEVICE(c);
  philox_probe_kernel<<<(n + 255) / 256, 256, 0, static_cast<cudaStream_t>(stream)>>>(
      c->p, reinterpret_cast<const uint4*>(d_ctr), n, reinterpret_cast<uint4*>(d_out));
  RA_CUDA(c, cudaGetLastError());
  return RA_OK;
}

ra_status ra_mppi_state_noise(ra_mppi_ctx* c, const int32_t* d_kmt, int32_t n, uint64_t iteration, float* d_w,
                              void* stream) {
  if (!c) return RA_EINVAL;
  if (!d_kmt || !d_w || n < 0) return fail(c, RA_EINVAL, "bad arguments");
  if (n == 0) return RA_OK;
  RA_ON_DEVICE(c);
  const Params p = with_iteration(c, iteration);
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  const int grid = (n + 255) / 256, nk = c->cfg.noise_kind;
#define RA_PROBE(NX, N) noise_probe_kernel<NX, N><<<grid, 256, 0, s>>>(p, d_kmt, n, d_w)
  if (p.nx == 4) { if (nk == 0) RA_PROBE(4, 0); else if (nk == 1) RA_PROBE(4, 1); else RA_PROBE(4, 2); }
  else { if (nk == 0) RA_PROBE(6, 0); else if (nk == 1) RA_PROBE(6, 1); else RA_PROBE(6, 2); }
#undef RA_PROBE
  RA_CUDA(c, cudaGetLastError());
  return RA_OK;
}

}  // extern "C"

namespace {
__global__ void set_loop_kernel(LoopState* loop, unsigned long long iter0) {
  loop->iter = iter0;
  loop->log_idx = 0ull;
}
}  // namespace

extern "C" {

ra_status ra_mppi_closed_loop(ra_mppi_ctx* c, float* d_x0, float* d_v, uint64_t iteration0, int32_t n_iter,
                              float* d_log, float* h_ms, void* stream) {
  if (!c) return RA_EINVAL;
  if (!d_x0 || !d_v || n_iter < 0) return fail(c, RA_EINVAL, "bad arguments");
  if (n_iter == 0) return RA_OK;
  RA_ON_DEVICE(c);
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  cudaStream_t own = nullptr;
  if (s == nullptr) {  // the legacy default stream cannot be captured
    // a blocking stream: ordered after (and before) the work the caller put on the NULL stream
    RA_CUDA(c, cudaStreamCreate(&own));
    s = own;
  }
  ra_status st = RA_OK;
  std::vector<cudaEvent_t> ev;
  do {
    // (re)capture one iteration: sampling, nominal || noisy rollouts, weights/update with the plant/shift tail, all reading
    // the device-resident counter
    if (!c->graph_exec || c->g_x0 != d_x0 || c->g_v != d_v || c->g_log != d_log) {
      if (c->graph_exec) { cudaGraphExecDestroy(c->graph_exec); c->graph_exec = nullptr; }
      Params p = c->p;
      p.d_iter = &c->d_loop->iter;
      p.iter_imm = 0;
      cudaGraph_t graph = nullptr;
      if (cudaStreamBeginCapture(s, cudaStreamCaptureModeThreadLocal) != cudaSuccess) { st = fail(c, RA_ECUDA, "begin capture"); break; }
      st = enqueue_costs(c, p, d_x0, d_v, nullptr, nullptr, s, false);
      // the last CTA of the weights/update kernel applies v+_0 to the plant and shifts v: no separate kernels
      if (st == RA_OK) st = enqueue_update(c, p, d_v, s, UpdateTail{d_x0, d_log, c->d_loop});
      cudaError_t e = cudaStreamEndCapture(s, &graph);
      if (st != RA_OK) { if (graph) cudaGraphDestroy(graph); break; }
      if (e != cudaSuccess) { st = cuda_fail(c, e, "end capture"); break; }
      e = cudaGraphInstantiate(&c->graph_exec, graph, 0);
      cudaGraphDestroy(graph);
      if (e != cudaSuccess) { c->graph_exec = nullptr; st = cuda_fail(c, e, "graph instantiate"); break; }
      c->g_x0 = d_x0; c->g_v = d_v; c->g_log = d_log;
    }
    set_loop_kernel<<<1, 1, 0, s>>>(c->d_loop, (unsigned long long)iteration0);
    if ((st = cuda_fail(c, cudaGetLastError(), "set_loop")) != RA_OK) break;
    if (h_ms) {
      ev.resize((size_t)n_iter + 1);
      for (auto& e : ev) if (cudaEventCreate(&e) != cudaSuccess) { st = fail(c, RA_ECUDA, "event create"); break; }
      if (st != RA_OK) break;
      cudaEventRecord(ev[0], s);
    }
    for (int i = 0; i < n_iter; ++i) {
      cudaError_t e = cudaGraphLaunch(c->graph_exec, s);
      if (e != cudaSuccess) { st = cuda_fail(c, e, "graph launch"); break; }
      if (h_ms) cudaEventRecord(ev[(size_t)i + 1], s);
    }
    if (st != RA_OK) break;
    if (h_ms || own) {
      cudaError_t e = cudaStreamSynchronize(s);
      if (e != cudaSuccess) { st = cuda_fail(c, e, "closed loop sync"); break; }
    }
    if (h_ms)
      for (int i = 0; i < n_iter; ++i) cudaEventElapsedTime(&h_ms[i], ev[(size_t)i], ev[(size_t)i + 1]);
  } while (false);
  for (auto e : ev) if (e) cudaEventDestroy(e);
  if (own) cudaStreamDestroy(own);
  return st;
}

}  // extern "C"

// =======================================================================================
// ra_mppi_weights_update_static: weights (17) and update (4) without a context and without any device allocation
// (include/ra_mppi.h says who needs that).  The kernel is the library's weights_update_kernel in its multi-range form:
// every CTA writes its range's {beta, Z, N_t} into `partial`, takes a ticket from `done`, and the last CTA combines the
// ranges.  Elsewhere those two buffers are cudaMalloc'ed by the context; here they are the array below.
//
// g_static_update_scratch is a __device__ variable: in HOST code its name is a stand-in the runtime uses to find the
// per-device instance, not a device address.  Handing `g_static_update_scratch` (or &g_static_update_scratch[0])
// to a kernel from host code would pass a host address: the kernel faults, or on a system where the GPU can read
// host memory quietly works on the wrong bytes.  The device address comes from cudaGetSymbolAddress, per device, with
// that device current (static_scratch_on_current_device below).
// =======================================================================================
namespace {
constexpr size_t kStaticPartialBytes = sizeof(double) * kMaxUpdateSplits * (2 + 2 * RA_MAX_T);
constexpr size_t kStaticTicketOffset = kStaticPartialBytes;            // the ticket sits behind the partial sums
constexpr size_t kStaticScratchBytes = kStaticPartialBytes + 256;
static_assert(kStaticScratchBytes == RA_STATIC_SCRATCH_BYTES, "include/ra_mppi.h states the size of the static scratch");
static_assert(kStaticTicketOffset % 256 == 0, "ticket slot keeps the array's alignment");
static_assert(RA_STATIC_MAX_K == kMaxUpdateSplits * kUpdateThreads * kUpdateCached,
              "the limit is what kMaxUpdateSplits register-cached ranges hold");
}  // namespace

static __device__ __align__(256) unsigned char g_static_update_scratch[kStaticScratchBytes];

namespace {

struct StaticScratchSlot {
  std::atomic<unsigned char*> base{nullptr};   // device address of g_static_update_scratch on this device
  std::atomic<int> n_sm{0};
};
StaticScratchSlot g_static_slot[kMaxDevices];

thread_local char g_static_error[256] = "";

ra_status static_fail(ra_status st, const char* what, const char* detail = "") {
  std::snprintf(g_static_error, sizeof g_static_error, "ra_mppi_weights_update_static: %s%s%s", what,
                detail[0] ? ": " : "", detail);
  return st;
}

// Once per device (ordinals past the table: every call): the array's address on the CURRENT device and its SM count.
// Neither call allocates; the first may make the runtime load this library's module onto the device.
ra_status static_scratch_on_current_device(unsigned char** base, int* n_sm) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return static_fail(RA_ECUDA, "cudaGetDevice", cudaGetErrorString(e));
  const bool cached = dev >= 0 && dev < kMaxDevices;
  if (cached) {
    unsigned char* b = g_static_slot[dev].base.load(std::memory_order_acquire);
    if (b) { *base = b; *n_sm = g_static_slot[dev].n_sm.load(std::memory_order_relaxed); return RA_OK; }
  }
  void* ptr = nullptr;
  e = cudaGetSymbolAddress(&ptr, g_static_update_scratch);
  if (e != cudaSuccess || !ptr)
    return static_fail(RA_ECUDA, "cudaGetSymbolAddress(g_static_update_scratch) (is the current device an sm_100 GPU?)",
                       cudaGetErrorString(e));
  int sms = 0;
  e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  if (e != cudaSuccess || sms < 1) return static_fail(RA_ECUDA, "cudaDeviceGetAttribute", cudaGetErrorString(e));
  if (cached) {
    g_static_slot[dev].n_sm.store(sms, std::memory_order_relaxed);
    g_static_slot[dev].base.store(static_cast<unsigned char*>(ptr), std::memory_order_release);
  }
  *base = static_cast<unsigned char*>(ptr);
  *n_sm = sms;
  return RA_OK;
}

}  // namespace

extern "C" {

ra_status ra_mppi_weights_update_static(int32_t K, int32_t T, float lambda, const float* u_min, const float* u_max,
                                        const float* d_S_tilde, const float* d_u, float* d_v_plus, void* stream) {
  g_static_error[0] = '\0';
  if (!u_min || !u_max || !d_S_tilde || !d_u || !d_v_plus) return static_fail(RA_EINVAL, "null pointer");
  if (K < 1 || T < 1) return static_fail(RA_EINVAL, "K and T must be at least 1");
  if (!(lambda > 0.0f) || !std::isfinite(lambda)) return static_fail(RA_EINVAL, "lambda must be positive and finite");
  for (int i = 0; i < 2; ++i)
    if (!(u_min[i] <= u_max[i])) return static_fail(RA_EINVAL, "u_min must not exceed u_max");
  if (K > RA_STATIC_MAX_K || T > RA_MAX_T) {
    char msg[160];
    std::snprintf(msg, sizeof msg, "K = %d, T = %d do not fit the %d-byte static scratch (K <= %d, T <= %d); use a context",
                  (int)K, (int)T, (int)RA_STATIC_SCRATCH_BYTES, (int)RA_STATIC_MAX_K, (int)RA_MAX_T);
    return static_fail(RA_EUNSUPPORTED, msg);
  }
  unsigned char* base = nullptr;
  int n_sm = 0;
  if (ra_status st = static_scratch_on_current_device(&base, &n_sm)) return st;
  double* partial = reinterpret_cast<double*>(base);
  unsigned int* done = reinterpret_cast<unsigned int*>(base + kStaticTicketOffset);

  Params p{};   // the kernel reads the sizes, the temperature and the clamp only (no closed-loop tail here)
  p.K = K; p.T = T;
  p.neg_log2e_over_lambda = (float)(-1.4426950408889634 / (double)lambda);
  for (int i = 0; i < 2; ++i) { p.u_min[i] = u_min[i]; p.u_max[i] = u_max[i]; }
  // ranges and steps per CTA as the context's update picks them: a range is what one CTA caches in registers
  const int per_cta = kUpdateThreads * kUpdateCached;
  const int splits = std::max(1, std::min(kMaxUpdateSplits, (K + per_cta - 1) / per_cta));
  const int steps = std::max(1, std::min(kUpdateMaxSteps, (T * splits) / (2 * n_sm)));
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  // the ticket must start at zero; the kernel's last CTA re-arms it, but a call that was aborted half way would not have
  cudaError_t e = cudaMemsetAsync(done, 0, sizeof(unsigned int), s);
  if (e != cudaSuccess) return static_fail(RA_ECUDA, "cudaMemsetAsync(ticket)", cudaGetErrorString(e));
  weights_update_kernel<float><<<dim3((T + steps - 1) / steps, splits), kUpdateThreads, 0, s>>>(
      p, d_S_tilde, nullptr, reinterpret_cast<const float2*>(d_u), (long long)T, 1LL, d_v_plus, nullptr, nullptr, partial,
      done, UpdateTail{nullptr, nullptr, nullptr}, steps);
  e = cudaGetLastError();
  if (e != cudaSuccess) return static_fail(RA_ECUDA, "kernel launch", cudaGetErrorString(e));
  return RA_OK;
}

const char* ra_mppi_weights_update_static_error(void) { return g_static_error; }

}  // extern "C"
