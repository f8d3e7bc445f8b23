// Rollout kernels of the RA-MPPI iteration (Alg.1 l.3-29).
//   sample_kernel         : A1       (parallel over (k, t))
//   nominal_kernel        : A2       (one thread per control sample k)
//   noisy_rollout_kernel  : A3 + A4 + A5 + A6 + A7 (one warp, or half-warp when M <= 16, per
//                           control sample; lanes over the M realisations; noise in registers)
#pragma once
#include "models.cuh"
#include "ra_params.cuh"
#include "rng.cuh"

namespace ra {

constexpr int kRolloutThreads = 256;
constexpr int kRolloutWarps = kRolloutThreads / 32;
constexpr int NOISE_MATERIALISED = 3;  // rollout-kernel variant that reads w from HBM

// ---------------------------------------------------------------------------------------
// A1.  eps^k_t = sigma_eps (.) z, u^k_t = (k < K0 ? v_t : 0) + eps^k_t   (2c) PAPER.md:42, Alg.1 l.4-10.
// Parallel over (k, t): Philox + accurate Box-Muller + tan / sincos of the clamped control, once per
// (k, t).  Writes u_raw[T][K] (for the update (4)) and the control effects ce[K][T] (for both rollouts).
// ---------------------------------------------------------------------------------------
constexpr int kSampleThreads = 256;
constexpr int kSampleKB = 16;  // control samples per CTA row: 16 consecutive k make one 128-byte segment of u_raw[t][.]

// One (k, t) draw per thread (the kernel is a dependent chain -- Philox, log, sqrt, tan -- so it is laid out for
// latency, not for work per thread): blockIdx.x picks 16 consecutive samples, blockIdx.y a chunk of their T * 16 draws.
template <int DYN>
__global__ void __launch_bounds__(kSampleThreads) sample_kernel(const __grid_constant__ Params p,
                                                                const float* __restrict__ v) {
  const int idx = blockIdx.y * kSampleThreads + threadIdx.x;
  const int t = idx / kSampleKB, k = blockIdx.x * kSampleKB + idx % kSampleKB;
  if (t >= p.T || k >= p.K) return;
  const uint4 r = philox4x32_10((uint32_t)(k + p.k_off), 0u, (uint32_t)t, iteration_field(p, STREAM_EPS), p.rk);
  float z0, z1;
  box_muller(r.x, r.y, z0, z1);
  const bool with_mean = k + p.k_off < p.K0;
  const float u0 = fmaf(p.sigma_eps[0], z0, with_mean ? __ldg(v + 2 * t) : 0.0f);
  const float u1 = fmaf(p.sigma_eps[1], z1, with_mean ? __ldg(v + 2 * t + 1) : 0.0f);
  RA_DEVICE_CHECK(t >= 0 && t < p.T && k >= 0 && k < p.K);
  p.u_raw[(size_t)t * p.K + k] = make_float2(u0, u1);
  p.ce[(size_t)k * p.T + t] = control_effect<DYN>(p, u0, u1);
}

// ---------------------------------------------------------------------------------------
// A2.  Nominal rollout and S_k = sum_t [q(x_t) + gamma v_t^T Sigma^-1 u_t] + phi(x_T)   (3) PAPER.md:47,
// Alg.1 l.11-15: one thread per control sample (the only sequential chain of the K*T work), full warps.
// S is accumulated in fp64 (K*T adds only) because the softmin weights of (17) are sensitive to
// absolute errors in S~.  Independent of the noisy rollouts, so ra_mppi_step runs it beside them.
// ---------------------------------------------------------------------------------------
constexpr int kNominalThreads = 64;

template <int DYN, int NOM>
__global__ void __launch_bounds__(kNominalThreads) nominal_kernel(const __grid_constant__ Params p,
                                                                  const float* __restrict__ x0g,
                                                                  const float* __restrict__ v) {
  constexpr int NX = StateDim<DYN>::value;
  pdl_launch_dependents();
  pdl_wait();                // baseline-MPPI steps (A = 0) launch this kernel as a dependent of the sampling kernel
  const int k = blockIdx.x * kNominalThreads + threadIdx.x;
  if (k >= p.K) return;
  const float x0X = x0g[0], x0Y = x0g[1];
  float x[NX];
  x[0] = 0.0f; x[1] = 0.0f;
#pragma unroll
  for (int i = 2; i < NX; ++i) x[i] = x0g[i];
  if constexpr (DYN == DYN_SINGLE_TRACK) x[3] = fmaxf(x[3], p.dyn_p[6]);
  const float4* ce_k = p.ce + (size_t)k * p.T;
  double S = 0.0;
  // The step is a dependent chain, and its inputs (u, ce: two L2 loads per step) do not depend on it: fetch them a block
  // of steps ahead, so the chain pays the load latency once per block instead of once per step (nominal kernel at
  // K = 16384, T = 50: 36 -> 22 us with the shorter cost chain, -> 11 us with the blocked loads).
  constexpr int kBlock = 8;
  for (int t0 = 0; t0 < p.T; t0 += kBlock) {
    float2 ub[kBlock];
    float4 cb[kBlock];
#pragma unroll
    for (int j = 0; j < kBlock; ++j) {
      const int t = min(t0 + j, p.T - 1);
      RA_DEVICE_CHECK(t >= 0 && t < p.T && k < p.K);
      ub[j] = p.u_raw[(size_t)t * p.K + k];
      cb[j] = ce_k[t];
    }
#pragma unroll
    for (int j = 0; j < kBlock; ++j) {
      const int t = t0 + j;
      if (t < p.T) {
        const float ctrl = fmaf(p.ctrl_w[0] * __ldg(v + 2 * t), ub[j].x, p.ctrl_w[1] * __ldg(v + 2 * t + 1) * ub[j].y);  // gamma v^T Sigma^-1 u  (3)
        const float q = nominal_cost<NOM>(p, x0X + x[0], x0Y + x[1], x[3]);
        S += (double)q + (double)ctrl;
        dynamics_step<DYN>(p, x, cb[j]);
      }
    }
  }
  S += (double)terminal_cost<NOM>(p, x0X + x[0], x0Y + x[1], x[3], x0X, x0Y);
  p.S[k] = S;
}

// order-preserving map float -> uint32 (larger float <=> larger key); 0 is below every float
__device__ __forceinline__ uint32_t float_key(float f) {
  const uint32_t b = __float_as_uint(f);
  return (b & 0x80000000u) ? ~b : (b | 0x80000000u);
}
__device__ __forceinline__ float key_float(uint32_t k) {
  return __uint_as_float((k & 0x80000000u) ? (k ^ 0x80000000u) : ~k);
}

template <int G>
__device__ __forceinline__ float group_sum(float v, uint32_t mask) {
#pragma unroll
  for (int o = G / 2; o > 0; o >>= 1) v += __shfl_xor_sync(mask, v, o);
  return v;
}

// ---------------------------------------------------------------------------------------
// A6: CVaR_k = mean of the k_tail largest of the M risk costs (Alg.1 l.25-26 PAPER.md:204-207,
// (12) :107) on order-preserving keys.  keys: R_total slots per lane in shared memory (slot r of
// lane l at keys[r*32 + l]; key 0 marks an unused slot).  Both selectors work on VALUES, so the
// result does not depend on which of several tied realisations are "picked".
//   radix: 32 rounds of (compare, warp REDUX) find the k_tail-th largest value exactly; the tail sum is
//          sum(values above it) + (k_tail - count above) * it.  Any k_tail, any R_total.
// Returns CVaR of the raw costs; *mean_out = (1/M) sum (for (18)-(19)) when want_mean.
// ---------------------------------------------------------------------------------------
template <int G>
__device__ __forceinline__ float cvar_select_radix(const uint32_t* keys, int R_total, int lane, int k_tail,
                                                   uint32_t mask) {
  uint32_t prefix = 0u;
  int k_rem = k_tail;
  for (int bit = 31; bit >= 0; --bit) {
    const uint32_t cand = (prefix | (1u << bit)) >> bit;
    int cnt = 0;
    for (int r = 0; r < R_total; ++r) cnt += ((keys[r * 32 + lane] >> bit) == cand) ? 1 : 0;
    cnt = __reduce_add_sync(mask, cnt);
    if (cnt >= k_rem) prefix |= (1u << bit); else k_rem -= cnt;
  }
  // prefix = key of the k_tail-th largest; k_rem = how many copies of it belong to the tail
  float sum_gt = 0.0f;
  for (int r = 0; r < R_total; ++r) {
    const uint32_t key = keys[r * 32 + lane];
    sum_gt += (key > prefix) ? key_float(key) : 0.0f;
  }
  sum_gt = group_sum<G>(sum_gt, mask);
  return fmaf((float)k_rem, key_float(prefix), sum_gt) / (float)k_tail;
}

// Small tails (k_tail <= kTopkMaxTail, at most kTopkSlots slots per lane: every BASELINE config):
// repeated max extraction on keys held in registers.  Each round takes the largest remaining value
// with one REDUX.MAX, counts its copies with one REDUX.ADD, adds min(copies, k_rem) of it to the tail sum
// and clears them -- at most k_tail rounds of ~4 instructions per slot, instead of 32 radix rounds.
constexpr int kTopkSlots = 8;       // M <= 256 with 32 lanes per sample
constexpr int kTopkMaxTail = 40;
template <int G>
__device__ __forceinline__ float cvar_select_topk(const uint32_t* keys, int R_total, int lane, int k_tail,
                                                  uint32_t mask) {
  uint32_t key[kTopkSlots];
#pragma unroll
  for (int r = 0; r < kTopkSlots; ++r) key[r] = (r < R_total) ? keys[r * 32 + lane] : 0u;
  float sum = 0.0f;
  int k_rem = k_tail;
  while (k_rem > 0) {
    uint32_t top = key[0];
#pragma unroll
    for (int r = 1; r < kTopkSlots; ++r) top = max(top, key[r]);
    top = __reduce_max_sync(mask, top);
    int cnt = 0;
#pragma unroll
    for (int r = 0; r < kTopkSlots; ++r) {
      const bool is_top = key[r] == top;
      cnt += is_top ? 1 : 0;
      key[r] = is_top ? 0u : key[r];
    }
    cnt = __reduce_add_sync(mask, cnt);
    const int take = min(cnt, k_rem);
    sum = fmaf((float)take, key_float(top), sum);
    k_rem -= take;
  }
  return sum / (float)k_tail;
}

template <int G>
__device__ __forceinline__ float cvar_select(const uint32_t* keys, int R_total, int lane, int k_tail,
                                             int M, uint32_t mask, bool want_mean, float* mean_out) {
  if (want_mean) {   // (18)-(19) need the sample mean only when B != 1
    float sum_all = 0.0f;
    for (int r = 0; r < R_total; ++r) {
      const uint32_t key = keys[r * 32 + lane];
      sum_all += key ? key_float(key) : 0.0f;
    }
    *mean_out = group_sum<G>(sum_all, mask) / (float)M;
  }
  if (R_total <= kTopkSlots && k_tail <= kTopkMaxTail) return cvar_select_topk<G>(keys, R_total, lane, k_tail, mask);
  return cvar_select_radix<G>(keys, R_total, lane, k_tail, mask);
}

// Warp-wide float min / max in one instruction: redux.sync.{min,max}.f32 (sm_100a; SASS CREDUX).
__device__ __forceinline__ float warp_min_f32(float v) {
  float r;
  asm volatile("redux.sync.min.f32 %0, %1, 0xffffffff;" : "=f"(r) : "f"(v));
  return r;
}
__device__ __forceinline__ float warp_max_f32(float v) {
  float r;
  asm volatile("redux.sync.max.f32 %0, %1, 0xffffffff;" : "=f"(r) : "f"(v));
  return r;
}

// Risk running cost l(x~) (9) PAPER.md:93 for RC interleaved realisations of one lane.
// RISK_CIRCLES accumulates the UNWEIGHTED sum of squared penetrations; the kernel applies the weight
// risk_p[0] once after the horizon loop.
template <int RISK, int RC, int NX>
__device__ __forceinline__ void risk_accumulate(const Params& p, const float4* circ_s, int n_circ_pad, int lane,
                                                const MapFrame& mf, float x0X, float x0Y, float yaw_turns,
                                                const float (&x)[RC][NX], float (&L)[RC]) {
  if constexpr (RISK == RISK_CIRCLES || RISK == RISK_NOMINAL) {
    // RISK_NOMINAL: l = q of the paper's racing costs: smooth part per lane, then the
    // indicator obstacle cost (22) through the same culled candidate loop as the hinge cost.
    if constexpr (RISK == RISK_NOMINAL) {
#pragma unroll
      for (int r = 0; r < RC; ++r) L[r] += racing_smooth_cost(p, x0X + x[r][0], x0Y + x[r][1]);
    }
    // Exact culling: the lanes of a warp share u^k and start together, so they stay within a
    // few metres.  Once per step the warp takes the bounding box of all its positions (four
    // warp-wide CREDUX.F32), each lane tests one obstacle of a 32-obstacle batch against the box, and
    // every lane then evaluates only the balloted candidates.  The box distance uses the same
    // subtract / FMA structure as the per-lane distance below and fp32 rounding is monotone, so
    // box_d2 <= d2 holds exactly for every lane: a culled obstacle contributes exactly 0.  The staged
    // list is padded to a multiple of 32 with records of R^2 = 0, which are never near.
    float lox = x[0][0], hix = x[0][0], loy = x[0][1], hiy = x[0][1];
#pragma unroll
    for (int r = 1; r < RC; ++r) {
      lox = fminf(lox, x[r][0]); hix = fmaxf(hix, x[r][0]);
      loy = fminf(loy, x[r][1]); hiy = fmaxf(hiy, x[r][1]);
    }
    lox = warp_min_f32(lox); hix = warp_max_f32(hix);
    loy = warp_min_f32(loy); hiy = warp_max_f32(hiy);
    for (int base = 0; base < n_circ_pad; base += 32) {
      RA_DEVICE_CHECK(base + lane < n_circ_pad);
      const float4 cb = circ_s[base + lane];  // (cx - x0X, cy - x0Y, r + margin, (r + margin)^2)
      const float ddx = fmaxf(fmaxf(lox - cb.x, cb.x - hix), 0.0f);
      const float ddy = fmaxf(fmaxf(loy - cb.y, cb.y - hiy), 0.0f);
      uint32_t cand = __ballot_sync(0xFFFFFFFFu, fmaf(ddx, ddx, ddy * ddy) < cb.w);
      while (cand) {
        RA_DEVICE_CHECK(base + __ffs(cand) - 1 < n_circ_pad);
        const float4 c = circ_s[base + __ffs(cand) - 1];  // broadcast
        cand &= cand - 1u;
        float d2[RC];
        bool hit = false;
#pragma unroll
        for (int r = 0; r < RC; ++r) {
          const float dx = x[r][0] - c.x, dy = x[r][1] - c.y;
          d2[r] = fmaf(dx, dx, dy * dy);
          hit = hit || (d2[r] < c.w);
        }
        if (__any_sync(0xFFFFFFFFu, hit)) {   // most candidates of the box touch no realisation
#pragma unroll
          for (int r = 0; r < RC; ++r) {
            if (d2[r] < c.w) {
              if constexpr (RISK == RISK_NOMINAL) {
                L[r] += p.nom_p[5];                                      // c2 * 1[d_i < r_i]  (22)
              } else {
                float d;
                asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(d) : "f"(d2[r]));  // 1 ulp; pen = R - d
                const float pen = c.z - d;
                L[r] = fmaf(pen, pen, L[r]);
              }
            }
          }
        }
      }
    }
  } else if constexpr (RISK == RISK_COSTMAP) {
#pragma unroll
    for (int r = 0; r < RC; ++r) L[r] += bilinear_weighted(p, mf, x[r][0], x[r][1]);
  } else {  // test-only linear risk: weight * x[index]
    const int idx = (int)p.risk_p[1];
#pragma unroll
    for (int r = 0; r < RC; ++r) {
      float val = 0.0f;
#pragma unroll
      for (int i = 0; i < NX; ++i) val = (i == idx) ? x[r][i] : val;
      val = (idx == 2) ? restore_yaw(val, yaw_turns) : val + ((idx == 0) ? x0X : ((idx == 1) ? x0Y : 0.0f));
      L[r] = fmaf(p.risk_p[0], val, L[r]);
    }
  }
}

// ---------------------------------------------------------------------------------------
// A3-A7.  HALF: two control samples per warp (G = 16 lanes each, M <= 16).
// Dynamic shared memory: [n_circles] float4 obstacle records, [samples per CTA][T] float4 control
// effects, then per warp R_total*32 keys.
// ---------------------------------------------------------------------------------------
// Resident CTAs per SM (register budget).  Measured on B200 (profiles/r1d): with four interleaved realisations
// per lane (RC = 4) the costmap kernel (127 registers) and the single-track kernels (123; they spill at 80) are
// faster with 2 CTAs/SM than with 3 CTAs of 80 registers (C3 0.458 -> 0.445 ms); the bicycle + circles kernels
// (87 registers at most) and everything with RC <= 2 are faster with 3 (C1, C4, M = 256 sweep points).
// Throughput-, not latency-bound: 4-6 CTAs/SM are slower everywhere.
template <int DYN, int RISK, int RC>
constexpr int rollout_min_ctas() {
  return (RC == 4 && (DYN == DYN_SINGLE_TRACK || RISK == RISK_COSTMAP)) ? 2 : 3;
}
template <int DYN, int RISK, int NOISE, int RC, bool HALF>
__global__ void __launch_bounds__(kRolloutThreads, rollout_min_ctas<DYN, RISK, RC>())
noisy_rollout_kernel(const __grid_constant__ Params p, const float* __restrict__ x0g,
                     float* __restrict__ L_out, float* __restrict__ xT_out) {
  constexpr int NX = StateDim<DYN>::value;
  constexpr int G = HALF ? 16 : 32;
  extern __shared__ float4 smem4[];
  float4* circ_s = smem4;
  constexpr bool kUsesCircles = (RISK == RISK_CIRCLES || RISK == RISK_NOMINAL);
  const int n_circ_s = kUsesCircles ? ((p.n_circles + 31) & ~31) : 0;   // padded to whole 32-obstacle batches
  // wps warps share one control sample when K alone cannot fill the GPU (small K, large M):
  // warp ws of the sample takes the realisation chunks ws, ws + wps, ...; the CVaR select runs in
  // warp 0 of the sample after a CTA barrier.
  // HALF (M <= 16): a sample needs only half a warp, so a warp carries 2 RC samples -- lanes 0-15 / 16-31 of
  // realisation slot r belong to samples 2r / 2r+1 of the warp -- and always has wps = 1.  (With one slot per lane the
  // per-step obstacle culling, ~120 warp-instructions whatever RC is, is spread over half as many state-steps.)
  const int wps = HALF ? 1 : p.wps;
  constexpr int kCeSlotsMax = HALF ? 2 * RC * kRolloutWarps : kRolloutWarps;
  const int ce_slots = HALF ? kCeSlotsMax : kRolloutWarps / wps;
  float4* ce_all = smem4 + n_circ_s;                                   // [ce_slots][T] control effects
  uint32_t* keys_all = reinterpret_cast<uint32_t*>(ce_all + (size_t)ce_slots * p.T);

  pdl_launch_dependents();   // the weights/update kernel may be scheduled behind the last wave of this grid
  // the three regions fit the dynamic shared memory the launcher asked for
  RA_DEVICE_CHECK((size_t)n_circ_s * sizeof(float4) + (size_t)ce_slots * p.T * sizeof(float4) +
                  (size_t)kRolloutWarps * (HALF ? RC : p.R_total) * 32 * sizeof(uint32_t) <= dynamic_smem_bytes());
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const float x0X = x0g[0], x0Y = x0g[1];

  const int sample_in_cta = warp / wps, ws = warp - sample_in_cta * wps;
  const int sample = blockIdx.x * (kRolloutWarps / wps) + sample_in_cta;
  const int sub = HALF ? (lane & 15) : lane;
  const uint32_t mask = HALF ? (0xFFFFu << (lane & 16)) : 0xFFFFFFFFu;
  // sample of realisation slot r of this lane: the warp's one sample, or (HALF) sample 2r + (lane >> 4) of the warp's 2 RC
  int k_of[RC];
  bool k_valid_of[RC];
  const float4* ce_of[RC];     // its control-effect row in shared memory
  uint32_t* keys_of[RC];       // its key row(s): [R_total][32], or (HALF) one row of 32 shared by the two samples of slot r
  int ce_slot_of[RC];
#pragma unroll
  for (int r = 0; r < RC; ++r) {
    const int k_raw = HALF ? ((blockIdx.x * kRolloutWarps + warp) * RC + r) * 2 + (lane >> 4) : sample;
    k_valid_of[r] = k_raw < p.K;
    k_of[r] = k_valid_of[r] ? k_raw : p.K - 1;
    ce_slot_of[r] = HALF ? (warp * RC + r) * 2 + (lane >> 4) : sample_in_cta;
    ce_of[r] = ce_all + (size_t)ce_slot_of[r] * p.T;
    RA_DEVICE_CHECK(ce_slot_of[r] >= 0 && ce_slot_of[r] < ce_slots && ce_slot_of[r] < kCeSlotsMax);
    keys_of[r] = keys_all + (HALF ? (size_t)(warp * RC + r) * 32 : (size_t)sample_in_cta * p.R_total * 32);
  }

  // The T control effects of sample k (one contiguous row of ce[K][T], 16 T bytes) go to shared memory once, so the step
  // loop reads them with a broadcast LDS instead of a dependent L2 load per step.  The row is moved by the TMA engine:
  // one thread per row arms an mbarrier with the byte count and issues a 1-D bulk copy (cp.async.bulk, SASS UBLKCP); the
  // copy runs while the CTA stages its obstacles, and the threads that use the row wait on the barrier's phase.
  // Measured against an LDG/STS loop per warp: C3 step 0.393 -> 0.387 ms, other workloads equal (profiles/r2_tma_experiment.md).
  __shared__ __align__(8) unsigned long long ce_bar[kCeSlotsMax];
  if (ws == 0 && sub == 0) {
#pragma unroll
    for (int r = 0; r < (HALF ? RC : 1); ++r) {
      const uint32_t bar = (uint32_t)__cvta_generic_to_shared(&ce_bar[ce_slot_of[r]]);
      const uint32_t dst = (uint32_t)__cvta_generic_to_shared(ce_of[r]);
      const uint32_t bytes = (uint32_t)p.T * (uint32_t)sizeof(float4);
      asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(bar));
      asm volatile("fence.mbarrier_init.release.cluster;");
      asm volatile("fence.proxy.async.shared::cta;");     // the barrier's initialisation is visible to the async proxy
      asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
      asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                   ::"r"(dst), "l"(p.ce + (size_t)k_of[r] * p.T), "r"(bytes), "r"(bar) : "memory");
    }
  }
  if constexpr (kUsesCircles) {
    for (int i = threadIdx.x; i < n_circ_s; i += blockDim.x) {
      float4 c = make_float4(0.0f, 0.0f, 0.0f, 0.0f);   // padding: R^2 = 0 is never near
      if (i < p.n_circles) {
        c = p.circles[i];
        c = make_float4(c.x - x0X, c.y - x0Y, c.z, c.z * c.z);
      }
      circ_s[i] = c;
    }
  }
  MapFrame mf{};
  if constexpr (RISK == RISK_COSTMAP) mf = make_map_frame(p, x0X, x0Y);

  __syncthreads();   // obstacles staged; the barriers are initialised for every thread that waits on one
#pragma unroll
  for (int r = 0; r < (HALF ? RC : 1); ++r) {
    const uint32_t bar = (uint32_t)__cvta_generic_to_shared(&ce_bar[ce_slot_of[r]]);
    asm volatile("{\n\t.reg .pred P1;\n\tRA_WAIT_CE:\n\tmbarrier.try_wait.parity.shared::cta.b64 P1, [%0], 0;\n\t@!P1 bra RA_WAIT_CE;\n\t}"
                 ::"r"(bar) : "memory");
  }

  float x_init[NX];
  x_init[0] = 0.0f; x_init[1] = 0.0f;
#pragma unroll
  for (int i = 2; i < NX; ++i) x_init[i] = x0g[i];
  if constexpr (DYN == DYN_SINGLE_TRACK) x_init[3] = fmaxf(x_init[3], p.dyn_p[6]);
  // the models see the yaw only through sin / cos: integrate it from [-pi, pi) and add the whole turns back on output
  float yaw_turns;
  x_init[2] = reduce_yaw(x_init[2], yaw_turns);

  const uint32_t c3 = iteration_field(p, STREAM_W);
  uint32_t kg[RC];                               // global sample index in the Philox counter
#pragma unroll
  for (int r = 0; r < RC; ++r) kg[r] = (uint32_t)(k_of[HALF ? r : 0] + p.k_off);

  for (int chunk = ws * RC; chunk < p.R_total; chunk += wps * RC) {
    float x[RC][NX], L[RC];
    uint32_t m[RC];
#pragma unroll
    for (int r = 0; r < RC; ++r) {
      L[r] = 0.0f;
      m[r] = HALF ? (uint32_t)sub : (uint32_t)((chunk + r) * G + sub);
#pragma unroll
      for (int i = 0; i < NX; ++i) x[r][i] = x_init[i];
    }
    // one transition of all RC realisations of this lane: l(x~_t) at the pre-step state, then
    // x~_{t+1} = F(x~_t, u_t) + w_t   (6) PAPER.md:63 with w_t = wscale (.) a
    auto advance = [&](int t, const float (&a)[RC][NX]) {
      float4 ce_shared;
      if constexpr (!HALF) ce_shared = ce_of[0][t];   // the slots share a sample: one broadcast LDS per step
      risk_accumulate<RISK, RC, NX>(p, circ_s, n_circ_s, lane, mf, x0X, x0Y, yaw_turns, x, L);
#pragma unroll
      for (int r = 0; r < RC; ++r) {
        float4 ce;
        if constexpr (HALF) ce = ce_of[r][t]; else ce = ce_shared;
        dynamics_step<DYN, true>(p, x[r], ce);
#pragma unroll
        for (int i = 0; i < NX; ++i)
          x[r][i] = (NOISE == NOISE_MATERIALISED) ? x[r][i] + a[r][i] : fmaf(p.wscale[i], a[r][i], x[r][i]);
        if constexpr (DYN == DYN_SINGLE_TRACK) x[r][3] = fmaxf(x[r][3], p.dyn_p[6]);
      }
    };
    if constexpr (NOISE == NOISE_MATERIALISED) {
      for (int t = 0; t < p.T; ++t) {
        float a[RC][NX];
#pragma unroll
        for (int r = 0; r < RC; ++r) {
          // a slot past R_total (RC does not divide the slot count) has m >= M_pad: clamp it into the row so
          // the load stays inside w_mat; the slot's results are discarded below
          const uint32_t mc = min(m[r], (uint32_t)(p.M_pad - 1));
          RA_DEVICE_CHECK(k_of[r] < p.K && t < p.T && (int)mc < p.M_pad);
          const float* wp = p.w_mat + (((size_t)k_of[r] * p.T + t) * NX) * p.M_pad + mc;
#pragma unroll
          for (int i = 0; i < NX; ++i) a[r][i] = __ldg(wp + (size_t)i * p.M_pad);
        }
        advance(t, a);
      }
    } else if constexpr (NoiseWords<NX, NOISE>::value == 2) {
      // n_x = 4: one Philox call serves two steps (16 bits per uniform, one word per Box-Muller pair)
      int t = 0;
      for (; t + 1 < p.T; t += 2) {
        uint32_t carry[RC][2];
        float a[RC][NX];
#pragma unroll
        for (int r = 0; r < RC; ++r) {
          const uint4 q = philox4x32_10(kg[r], m[r], (uint32_t)(t >> 1), c3, p.rk);
          const uint32_t w[2] = {q.x, q.y};
          carry[r][0] = q.z; carry[r][1] = q.w;
          noise_from_words<NX, NOISE>(p, w, a[r]);
        }
        advance(t, a);
#pragma unroll
        for (int r = 0; r < RC; ++r) {
          const uint32_t w[2] = {carry[r][0], carry[r][1]};
          noise_from_words<NX, NOISE>(p, w, a[r]);
        }
        advance(t + 1, a);
      }
      if (t < p.T) {   // odd horizon: the last (even-indexed) step takes the first half of its call
        float a[RC][NX];
#pragma unroll
        for (int r = 0; r < RC; ++r) state_noise<NX, NOISE>(p, kg[r], m[r], (uint32_t)t, c3, a[r]);
        advance(t, a);
      }
    } else if constexpr (NoiseWords<NX, NOISE>::value == 3) {
      // three words per step (n_x = 6, or n_x = 4 with the jump trigger): three calls serve four steps
      int t = 0;
      for (; t + 3 < p.T; t += 4) {
        const uint32_t c = 3u * (uint32_t)(t >> 2);
        uint32_t carry[RC][3];
        float a[RC][NX];
#pragma unroll
        for (int r = 0; r < RC; ++r) {
          const uint4 qa = philox4x32_10(kg[r], m[r], c, c3, p.rk);
          const uint32_t w[3] = {qa.x, qa.y, qa.z};
          carry[r][0] = qa.w;
          noise_from_words<NX, NOISE>(p, w, a[r]);
        }
        advance(t, a);
#pragma unroll
        for (int r = 0; r < RC; ++r) {
          const uint4 qb = philox4x32_10(kg[r], m[r], c + 1u, c3, p.rk);
          const uint32_t w[3] = {carry[r][0], qb.x, qb.y};
          carry[r][0] = qb.z; carry[r][1] = qb.w;
          noise_from_words<NX, NOISE>(p, w, a[r]);
        }
        advance(t + 1, a);
#pragma unroll
        for (int r = 0; r < RC; ++r) {
          const uint4 qc = philox4x32_10(kg[r], m[r], c + 2u, c3, p.rk);
          const uint32_t w[3] = {carry[r][0], carry[r][1], qc.x};
          carry[r][0] = qc.y; carry[r][1] = qc.z; carry[r][2] = qc.w;
          noise_from_words<NX, NOISE>(p, w, a[r]);
        }
        advance(t + 2, a);
#pragma unroll
        for (int r = 0; r < RC; ++r) {
          const uint32_t w[3] = {carry[r][0], carry[r][1], carry[r][2]};
          noise_from_words<NX, NOISE>(p, w, a[r]);
        }
        advance(t + 3, a);
      }
      for (; t < p.T; ++t) {   // up to three ragged steps on their own
        float a[RC][NX];
#pragma unroll
        for (int r = 0; r < RC; ++r) state_noise<NX, NOISE>(p, kg[r], m[r], (uint32_t)t, c3, a[r]);
        advance(t, a);
      }
    } else {
      for (int t = 0; t < p.T; ++t) {
        float a[RC][NX];
#pragma unroll
        for (int r = 0; r < RC; ++r) state_noise<NX, NOISE>(p, kg[r], m[r], (uint32_t)t, c3, a[r]);
        advance(t, a);
      }
    }
#pragma unroll
    for (int r = 0; r < RC; ++r) {
      const bool slot_ok = HALF || (chunk + r) < p.R_total;
      const bool valid = slot_ok && (int)m[r] < p.M;
      if constexpr (RISK == RISK_CIRCLES) L[r] *= p.risk_p[0];   // risk_accumulate sums unweighted penetrations
      RA_DEVICE_CHECK(!slot_ok || (keys_of[r] + (HALF ? 0 : (chunk + r) * 32) + lane <
                                   keys_all + (size_t)kRolloutWarps * (HALF ? RC : p.R_total) * 32));
      if (slot_ok) keys_of[r][(HALF ? 0 : (chunk + r) * 32) + lane] = valid ? float_key(L[r]) : 0u;
      if (valid && k_valid_of[r]) {
        const int k = k_of[r];
        RA_DEVICE_CHECK(k >= 0 && k < p.K && (int)m[r] < p.M);
        if (L_out) L_out[(size_t)k * p.M + m[r]] = L[r];
        if (xT_out) {
          float* o = xT_out + ((size_t)k * p.M + m[r]) * NX;
          o[0] = x0X + x[r][0]; o[1] = x0Y + x[r][1];
          o[2] = restore_yaw(x[r][2], yaw_turns);
#pragma unroll
          for (int i = 3; i < NX; ++i) o[i] = x[r][i];
        }
      }
    }
  }
  if (wps > 1) {
    __syncthreads();          // every warp of the CTA reaches this exactly once (trip counts may differ)
    if (ws != 0) return;      // warp 0 of the sample reduces
  } else {
    __syncwarp();
  }

#pragma unroll
  for (int r = 0; r < (HALF ? RC : 1); ++r) {   // HALF: the two samples of every slot; otherwise the warp's one sample
    float Lbar = 0.0f;
    float cvar = cvar_select<G>(keys_of[r], p.R_total, lane, p.k_tail, p.M, mask, p.B != 1.0f, &Lbar);
    // (18)-(19) PAPER.md:144-148: L_a = B (L - Lbar) + Lbar is affine-monotone for B > 0, so
    // CVaR(L_a) = B (CVaR(L) - Lbar) + Lbar.
    if (p.B != 1.0f) cvar = fmaf(p.B, cvar - Lbar, Lbar);
    if (sub == 0 && k_valid_of[r]) {
      // soft filter (14)-(16) PAPER.md:120-130, strict threshold (15)
      RA_DEVICE_CHECK(k_of[r] >= 0 && k_of[r] < p.K);
      p.cvar[k_of[r]] = cvar;
      p.pen[k_of[r]] = (cvar > p.C_u) ? (double)(p.A * cvar) : 0.0;   // J_C of (14); S~ = S + J_C is formed by its readers
    }
  }
}

}  // namespace ra
