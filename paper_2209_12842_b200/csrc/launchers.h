// Host-side launch entry points of the per-(dynamics, risk) rollout translation units.
// rollout_inst.cu is compiled once per (RA_INST_DYN, RA_INST_RISK) pair so the template
// instantiations build in parallel; ra_mppi.cu picks the launcher at ra_mppi_create.
#pragma once
#include <cuda_runtime.h>

#include <atomic>

#include "ra_params.cuh"

namespace ra {

// cudaFuncSetAttribute acts on the CURRENT device's copy of a kernel, so "already set" is remembered per
// (kernel, device): `slot` is a zero-initialised static array of kMaxDevices entries owned by the call site
// (one per kernel instantiation) holding value + 1.  Ordinals past the table are simply set every time.
// A racing second thread at worst repeats the call.
constexpr int kMaxDevices = 64;
template <typename Kernel>
inline cudaError_t set_func_attr_once(std::atomic<int>* slot, int device, Kernel kernel, cudaFuncAttribute attr,
                                      int value) {
  const bool cached = device >= 0 && device < kMaxDevices;
  if (cached && slot[device].load(std::memory_order_relaxed) == value + 1) return cudaSuccess;
  const cudaError_t e = cudaFuncSetAttribute(kernel, attr, value);
  if (e == cudaSuccess && cached) slot[device].store(value + 1, std::memory_order_relaxed);
  return e;
}

// Kernel launch with or without programmatic dependent launch (PDL): with `pdl` the kernel may be scheduled while
// the previous kernel of the stream is still draining (after all its CTAs have executed griddepcontrol.launch_dependents
// or exited) and must execute griddepcontrol.wait before it touches that kernel's results.  Works in eager streams and
// under stream capture (the edge becomes a programmatic graph edge).
template <typename... KArgs, typename... Args>
inline cudaError_t launch_kernel(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t stream,
                                 bool pdl, Args&&... args) {
  cudaLaunchConfig_t cfg{};
  cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = stream;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = pdl ? 1u : 0u;
  return cudaLaunchKernelEx(&cfg, kernel, KArgs(args)...);
}

// noise: NOISE_GAUSSIAN / NOISE_UNIFORM / NOISE_JUMP / 3 (materialised); rc in {1,2,4};
// half: half a warp per sample (M <= 16; rc in {1,2} = 2 rc samples per warp); pdl: launch as a programmatic dependent of the
// previous kernel.
using RolloutLaunchFn = cudaError_t (*)(const Params& p, int noise, int rc, bool half, const float* d_x0,
                                        float* d_L, float* d_xT, cudaStream_t stream, bool pdl);

#define RA_DECLARE_ROLLOUT(D, R) \
  cudaError_t launch_rollout_##D##_##R(const Params& p, int noise, int rc, bool half, const float* d_x0, \
                                       float* d_L, float* d_xT, cudaStream_t stream, bool pdl);
RA_DECLARE_ROLLOUT(0, 0)
RA_DECLARE_ROLLOUT(0, 1)
RA_DECLARE_ROLLOUT(0, 2)
RA_DECLARE_ROLLOUT(0, 3)
RA_DECLARE_ROLLOUT(1, 0)
RA_DECLARE_ROLLOUT(1, 1)
RA_DECLARE_ROLLOUT(1, 2)
RA_DECLARE_ROLLOUT(1, 3)
#undef RA_DECLARE_ROLLOUT

}  // namespace ra
