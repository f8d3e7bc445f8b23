// Instantiates noisy_rollout_kernel for one (dynamics, risk) pair:
//   nvcc -DRA_INST_DYN=<0|1> -DRA_INST_RISK=<0|1|2> -c rollout_inst.cu
#include "../../include/ra_mppi.h"
#include "launchers.h"
#include "rollout.cuh"

#ifndef RA_INST_DYN
#error "define RA_INST_DYN"
#endif
#ifndef RA_INST_RISK
#error "define RA_INST_RISK"
#endif

namespace ra {
namespace {

template <int NOISE, int RC, bool HALF>
cudaError_t launch(const Params& p, const float* d_x0, float* d_L, float* d_xT, cudaStream_t stream, bool pdl) {
  const int samples_per_cta = HALF ? 2 * RC * kRolloutWarps : kRolloutWarps / p.wps;
  const int grid = (p.K + samples_per_cta - 1) / samples_per_cta;
  const int ce_slots = samples_per_cta;
  const int key_rows = kRolloutWarps * (HALF ? RC : p.R_total);
  const size_t smem = ((RA_INST_RISK == RISK_CIRCLES || RA_INST_RISK == RISK_NOMINAL) ? (size_t)((p.n_circles + 31) & ~31) * sizeof(float4) : 0) +
                      (size_t)ce_slots * p.T * sizeof(float4) + (size_t)key_rows * 32 * sizeof(uint32_t);
  auto kernel = noisy_rollout_kernel<RA_INST_DYN, RA_INST_RISK, NOISE, RC, HALF>;
  // Worst case over everything ra_mppi_create / ra_mppi_set_env accept: M <= 16 with two slots per lane (K >= 32768) stages
  // 32 control-effect rows, at T = 128 that is 64 KB, plus 2 KB of keys and 16 KB for 1024 circles = 82 KB; the other
  // layouts stay below 49 KB.  kRolloutSmemLimit covers that with room to spare (an SM holds 227 KB: two such CTAs fit).
  constexpr int kRolloutSmemLimit = 96 * 1024;
  static_assert((size_t)kMaxCirclesSmem * sizeof(float4) + (size_t)4 * kRolloutWarps * RA_MAX_T * sizeof(float4) +
                    (size_t)kRolloutWarps * (RA_MAX_M / 32) * 32 * sizeof(uint32_t) <= (size_t)kRolloutSmemLimit,
                "the largest accepted configuration must fit the dynamic shared-memory limit");
  if (smem > (size_t)kRolloutSmemLimit) return cudaErrorInvalidConfiguration;
  if (smem > 48 * 1024) {
    static std::atomic<int> smem_set[kMaxDevices];
    const cudaError_t e = set_func_attr_once(smem_set, p.device, kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kRolloutSmemLimit);
    if (e != cudaSuccess) return e;
  }
  // the same L1 / shared-memory split as the nominal-rollout kernel that runs beside this one: CTAs of kernels
  // with different carveouts do not share an SM (measured: +20 us per closed-loop iteration otherwise)
  static std::atomic<int> carveout_set[kMaxDevices];
  if (const cudaError_t e = set_func_attr_once(carveout_set, p.device, kernel, cudaFuncAttributePreferredSharedMemoryCarveout, p.carveout))
    return e;
  return launch_kernel(kernel, dim3(grid), dim3(kRolloutThreads), smem, stream, pdl, p, d_x0, d_L, d_xT);
}

template <int NOISE>
cudaError_t launch_noise(const Params& p, int rc, bool half, const float* d_x0, float* d_L, float* d_xT,
                         cudaStream_t stream, bool pdl) {
  if (half) {   // M <= 16: half a warp per sample, 2 rc samples per warp
    if (rc == 2) return launch<NOISE, 2, true>(p, d_x0, d_L, d_xT, stream, pdl);
    return rc == 1 ? launch<NOISE, 1, true>(p, d_x0, d_L, d_xT, stream, pdl) : cudaErrorInvalidValue;
  }
  switch (rc) {
    case 1: return launch<NOISE, 1, false>(p, d_x0, d_L, d_xT, stream, pdl);
    case 2: return launch<NOISE, 2, false>(p, d_x0, d_L, d_xT, stream, pdl);
    case 4: return launch<NOISE, 4, false>(p, d_x0, d_L, d_xT, stream, pdl);
    default: return cudaErrorInvalidValue;
  }
}

}  // namespace

#define RA_CAT2(a, b, c) launch_rollout_##a##_##b
#define RA_CAT(a, b) RA_CAT2(a, b, _)

cudaError_t RA_CAT(RA_INST_DYN, RA_INST_RISK)(const Params& p, int noise, int rc, bool half,
                                               const float* d_x0, float* d_L, float* d_xT,
                                               cudaStream_t stream, bool pdl) {
  switch (noise) {
    case NOISE_GAUSSIAN: return launch_noise<NOISE_GAUSSIAN>(p, rc, half, d_x0, d_L, d_xT, stream, pdl);
    case NOISE_UNIFORM: return launch_noise<NOISE_UNIFORM>(p, rc, half, d_x0, d_L, d_xT, stream, pdl);
    case NOISE_JUMP: return launch_noise<NOISE_JUMP>(p, rc, half, d_x0, d_L, d_xT, stream, pdl);
    case NOISE_MATERIALISED: return launch_noise<NOISE_MATERIALISED>(p, rc, half, d_x0, d_L, d_xT, stream, pdl);
    default: return cudaErrorInvalidValue;
  }
}

}  // namespace ra
