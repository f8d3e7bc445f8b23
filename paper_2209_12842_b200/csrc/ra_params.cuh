// Kernel-side parameter block of the RA-MPPI hot path (sm_100a).
// Built once per context on the host (ra_mppi.cu) and passed to every kernel by value.
#pragma once
#include <cstdint>
#include <cstdio>

// Bounds checks of the checked build (python -m paper_2209_12842_b200.build --checked -> libra_mppi_checked.so, used by
// tests/test_gpu_checked_build.py): compute-sanitizer is closed on the GPU pool, so the kernels carry their own index
// assertions, compiled out of the product library.  A failed check prints its condition and traps the kernel.
#ifdef RA_CHECKED
#define RA_DEVICE_CHECK(cond)                                                                   \
  do {                                                                                          \
    if (!(cond)) {                                                                              \
      printf("RA_DEVICE_CHECK failed: %s (%s:%d) block %d thread %d\n", #cond, __FILE__, __LINE__, \
             (int)blockIdx.x, (int)threadIdx.x);                                                \
      __trap();                                                                                 \
    }                                                                                           \
  } while (0)
#else
#define RA_DEVICE_CHECK(cond) do { } while (0)
#endif

namespace ra {

enum : int { DYN_BICYCLE = 0, DYN_SINGLE_TRACK = 1 };
enum : int { NOM_GOAL = 0, NOM_TRACK = 1, NOM_RACING = 2 };
enum : int { RISK_CIRCLES = 0, RISK_COSTMAP = 1, RISK_LINEAR = 2, RISK_NOMINAL = 3 };
enum : int { NOISE_GAUSSIAN = 0, NOISE_UNIFORM = 1, NOISE_JUMP = 2 };
enum : uint32_t { STREAM_EPS = 0u, STREAM_W = 1u, STREAM_PLANT = 2u };

constexpr int kMaxCirclesSmem = 1024;  // obstacle records staged per CTA (16 B each)

struct Params {
  int K, M, T;
  int K0;       // samples with GLOBAL index < K0 use u = v + eps, the rest u = eps   (Alg.1 l.7-10)
  int k_off;    // global index of local sample 0 (K-sharding; 0 when not sharded)
  int k_tail;   // ceil((1-alpha) M)                                  (Alg.1 l.25)
  int G;        // lanes per control sample: 32, or 16 when M <= 16
  int R_total;  // realisation slots of G lanes per sample = ceil(M / G)
  int wps;      // warps per control sample in the rollout kernel (1, 2, 4 or 8)
  int nx;
  int dyn, noise_kind;  // model and noise kind (runtime copies for the kernels that are not templated on them)
  int carveout; // host only: preferred shared-memory carveout (percent) of the two concurrent rollout kernels
  int device;   // host only: CUDA device ordinal of the context (per-device kernel attributes)
  float dt;
  float dyn_p[8];
  float dyn_q[2];   // single-track: 1/m, 1/Iz; bicycle: dt/L
  float u_min[2], u_max[2];
  float sigma_eps[2];
  float ctrl_w[2];  // gamma / sigma_eps^2 (0 where sigma_eps == 0)   (3) PAPER.md:47
  float sigma_w[6];
  float wscale[6];   // additive noise of (6): w_i = wscale[i] * a_i, a = state_noise() (rng.cuh)
  float neg_log2e_over_lambda;  // weights (17) PAPER.md:134 as exp2
  float A, B, C_u;
  float nom_p[12];
  float nom_q[2];   // ellipse track: 1/a, 1/b
  float risk_p[4];
  float noise_p[4];
  uint32_t rk[20];  // the ten Philox round keys (k0_r, k1_r), key = seed
  // environment (device copies owned by the context)
  const float4* circles;  // [n] absolute (cx, cy, r + risk margin, r)
  int n_circles;
  const float4* quadmap;  // [(map_h+1)][(map_w+1)] texel quads, clamp-to-edge baked in
  int map_h, map_w;
  float map_inv_res, map_ox, map_oy;
  // scratch owned by the context
  float2* u_raw;   // [T][K] sampled controls u^k_t (unclamped)
  float4* ce;      // [K][T] control effects consumed by the rollout kernels
  double* S;        // [K] nominal cost (3), fp64 so weight errors come from q, not from the sum
  float* cvar;      // [K]
  double* pen;      // [K] soft-filter term J_C of (14); the modified cost (16) is S + pen
  const float* w_mat;  // materialised noise [K][T][nx][M_pad] or nullptr
  int M_pad;
  // iteration index: device-resident when replayed from a graph, immediate otherwise
  const unsigned long long* d_iter;
  unsigned long long iter_imm;
};

// Programmatic dependent launch (launchers.h: launch_kernel): a kernel started early waits here for the previous
// kernel of its stream to finish and flush; a kernel lets its successor start being scheduled once every CTA has
// passed launch_dependents.  Both are no-ops for plain launches.
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;"); }

__device__ __forceinline__ uint32_t dynamic_smem_bytes() {
  uint32_t n;
  asm("mov.u32 %0, %%dynamic_smem_size;" : "=r"(n));
  return n;
}

__device__ __forceinline__ uint32_t iteration_field(const Params& p, uint32_t stream) {
  const unsigned long long it = p.d_iter ? *p.d_iter : p.iter_imm;
  return (stream << 28) | (uint32_t)(it & 0x0FFFFFFFull);
}

}  // namespace ra
