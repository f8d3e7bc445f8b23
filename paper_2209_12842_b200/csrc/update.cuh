// Weights (17)/(5), update (4), and the closed-loop glue (Alg.1 l.31-33).
#pragma once
#include "models.cuh"
#include "ra_params.cuh"
#include "rng.cuh"

namespace ra {

constexpr int kUpdateThreads = 256;   // small CTAs: 64 registers each (samples cached in registers), several per SM, one wave
constexpr int kUpdateCached = 8;      // samples per thread held in registers across the min reduction

template <typename T, typename Op>
__device__ __forceinline__ T block_reduce(T v, T* smem, Op op, T identity) {
  // fixed-order tree: xor-shuffle inside each warp, then warp 0 over the per-warp partials
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = op(v, __shfl_xor_sync(0xFFFFFFFFu, v, o));
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  __syncthreads();  // smem may still be read from a previous reduction
  if (lane == 0) smem[warp] = v;
  __syncthreads();
  v = (lane < (blockDim.x >> 5)) ? smem[lane] : identity;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = op(v, __shfl_xor_sync(0xFFFFFFFFu, v, o));
  return v;  // every thread holds the result
}

// Device-resident loop state for graph replay.
struct LoopState {
  unsigned long long iter;     // Philox iteration index of the next step
  unsigned long long log_idx;  // row of the closed-loop log to write next
};

// ---------------------------------------------------------------------------------------
// A10.  ExecuteCommand(v+_0) on the simulated plant (the disturbed dynamics (6) with the PLANT stream),
// v <- shift(v+) (Alg.1 l.32-33 PAPER.md:218-220 + BASELINE config 4's warm-start shift), iteration++.
// Executed by ONE CTA, all of its threads (it synchronises): the body of plant_shift_kernel and the tail of the
// weights/update kernel inside the captured closed loop, so both give the same bits.
// ---------------------------------------------------------------------------------------
template <int DYN, int NOISE>
__device__ __forceinline__ void plant_shift_cta(const Params& p, float* x0g, float* v, float* u_applied, float* log,
                                                LoopState* loop) {
  constexpr int NX = StateDim<DYN>::value;
  // shift: read everything, then write (T <= RA_MAX_T = 128 <= 2 * blockDim for every caller)
  float2 nxt[2];
  float2* v2 = reinterpret_cast<float2*>(v);
  int cnt = 0;
  for (int t = threadIdx.x; t < p.T && cnt < 2; t += blockDim.x) nxt[cnt++] = v2[min(t + 1, p.T - 1)];
  const float2 v0 = v2[0];
  __syncthreads();
  cnt = 0;
  for (int t = threadIdx.x; t < p.T && cnt < 2; t += blockDim.x) v2[t] = nxt[cnt++];

  if (threadIdx.x == 0) {
    float x[NX];
    const float x0X = x0g[0], x0Y = x0g[1];
    x[0] = 0.0f; x[1] = 0.0f;
#pragma unroll
    for (int i = 2; i < NX; ++i) x[i] = x0g[i];
    if constexpr (DYN == DYN_SINGLE_TRACK) x[3] = fmaxf(x[3], p.dyn_p[6]);
    const float4 ce = control_effect<DYN>(p, v0.x, v0.y);
    float z[NX];
    state_noise<NX, NOISE>(p, 0u, 0u, 0u, iteration_field(p, STREAM_PLANT), z);
    dynamics_step<DYN>(p, x, ce);
#pragma unroll
    for (int i = 0; i < NX; ++i) x[i] = fmaf(p.wscale[i], z[i], x[i]);
    if constexpr (DYN == DYN_SINGLE_TRACK) x[3] = fmaxf(x[3], p.dyn_p[6]);
    x[0] += x0X; x[1] += x0Y;
#pragma unroll
    for (int i = 0; i < NX; ++i) x0g[i] = x[i];
    if (u_applied) { u_applied[0] = v0.x; u_applied[1] = v0.y; }
    if (log) {
      float* row = log + (loop ? loop->log_idx : 0ull) * (NX + 2);
#pragma unroll
      for (int i = 0; i < NX; ++i) row[i] = x[i];
      row[NX] = v0.x; row[NX + 1] = v0.y;
    }
    if (loop) { loop->iter += 1ull; loop->log_idx += 1ull; }
  }
}

// the same, picking the (model, noise kind) instantiation at run time
__device__ __noinline__ void plant_shift_any(const Params& p, float* x0g, float* v, float* u_applied, float* log,
                                             LoopState* loop) {
  switch (p.dyn * 3 + p.noise_kind) {
    case 0: plant_shift_cta<0, 0>(p, x0g, v, u_applied, log, loop); break;
    case 1: plant_shift_cta<0, 1>(p, x0g, v, u_applied, log, loop); break;
    case 2: plant_shift_cta<0, 2>(p, x0g, v, u_applied, log, loop); break;
    case 3: plant_shift_cta<1, 0>(p, x0g, v, u_applied, log, loop); break;
    case 4: plant_shift_cta<1, 1>(p, x0g, v, u_applied, log, loop); break;
    default: plant_shift_cta<1, 2>(p, x0g, v, u_applied, log, loop); break;
  }
}

__global__ void __launch_bounds__(128) plant_shift_kernel(const __grid_constant__ Params p, float* x0g, float* v,
                                                          float* u_applied, float* log, LoopState* loop) {
  plant_shift_any(p, x0g, v, u_applied, log, loop);
}

// Exchange step of (17)/(4) over sample ranges or shards: partials [n][2+2T] = {beta_g, Z_g, N_g[T][2]}
// -> v+ = clamp(sum_g s_g N_g / sum_g s_g Z_g), s_g = exp(-(beta_g - beta)/lambda), beta = min_g beta_g,
// which is (17)/(4) over the union of the parts (factor exp(-(beta_g-beta)/lambda) out of every w~_k).
// Fixed summation order over g => every rank / every replay computes bitwise the same v+; fp64 until the final
// divide.  Executed by one CTA, thread = (t, i).  The partials may have been written by other CTAs of the running
// grid, hence the L2 loads (__ldcg).
__device__ __forceinline__ void combine_partials_cta(const Params& p, const double* partials, int n_parts,
                                                     float* v_out) {
  const int stride = 2 + 2 * p.T;
  double beta = INFINITY;
  for (int g = 0; g < n_parts; ++g) beta = fmin(beta, __ldcg(partials + (size_t)g * stride));
  for (int j = threadIdx.x; j < 2 * p.T; j += blockDim.x) {
    double Z = 0.0, n = 0.0;
    for (int g = 0; g < n_parts; ++g) {
      const double* pg = partials + (size_t)g * stride;
      const double s = (double)exp2f((float)(__ldcg(pg) - beta) * p.neg_log2e_over_lambda);
      Z = fma(s, __ldcg(pg + 1), Z);
      n = fma(s, __ldcg(pg + 2 + j), n);
    }
    v_out[j] = clampf((float)(n / Z), p.u_min[j & 1], p.u_max[j & 1]);
  }
}

__global__ void combine_partials_kernel(const __grid_constant__ Params p, const double* __restrict__ partials,
                                        int n_parts, float* __restrict__ v_out) {
  combine_partials_cta(p, partials, n_parts, v_out);
}

// ---------------------------------------------------------------------------------------
// A8 + A9.  One CTA per (group of steps_per_cta horizon steps, sample range blockIdx.y of gridDim.y).  Each CTA forms
// beta~ = min_k S~_k over its range (values from L2), w~_k = exp(-(S~_k - beta~)/lambda) and Z = sum w~ ONCE, then
// N_t = sum_k w~_k u^k_t for each of its steps   (17) PAPER.md:134, (5) :55, (4) :51.  The host picks the ranges (what a CTA
// caches in registers) and then the group size so that the grid is about two CTAs per SM: at large K this stops every
// step's CTA from re-reading the range's costs (K = 65536: 50 re-reads -> 9).  Three uses:
//   * ra_mppi_step: the CTA writes its range's {beta, Z, N_t} into `partial` (context scratch); the LAST CTA of the grid
//     to finish (an atomic ticket in *done) combines the ranges into v+ = clamp(N / Z) -- in a fixed order, so the
//     result does not depend on which CTA that was -- and, inside the captured closed loop (tail.x0g != nullptr), goes on
//     to apply v+_0 to the plant and shift v (A10): one kernel instead of three on the latency path of an iteration;
//   * ra_mppi_step_partial (K-sharded step): `partial` is the caller's, done == nullptr: the CTA just writes its share;
//   * ra_mppi_weights_update (caller's S~ and u, gridDim.y = 1, partial == nullptr): the CTA writes v+_t itself.
// u is addressed as u[k*su_k + t*su_t] so both the internal [T][K] scratch and a caller's [K][T] array work.
// Reduction order is fixed => bitwise reproducible.
// ---------------------------------------------------------------------------------------
// S~_k (16): the caller's array (ST = float), or S + J_C from the context scratch (ST = double, pen != nullptr)
template <typename ST>
__device__ __forceinline__ ST s_tilde_at(const ST* __restrict__ S, const double* __restrict__ pen, int k) {
  if constexpr (sizeof(ST) == sizeof(double)) return pen ? S[k] + pen[k] : S[k];
  else return S[k];
}

struct UpdateTail {          // closed-loop tail of the update kernel (all null outside ra_mppi_closed_loop)
  float* x0g;                // [n_x] state, advanced by the plant
  float* log;                // closed-loop log or nullptr
  LoopState* loop;
};

constexpr int kUpdateMaxSteps = 8;    // horizon steps one CTA may take (its samples' weights are formed once and reused)

template <typename ST>
__global__ void __launch_bounds__(kUpdateThreads)
weights_update_kernel(const __grid_constant__ Params p, const ST* __restrict__ S_tilde,
                      const double* __restrict__ pen, const float2* __restrict__ u, long long su_k, long long su_t,
                      float* v_out, float* __restrict__ w_out, float* __restrict__ stats, double* partial,
                      unsigned int* done, UpdateTail tail, int steps_per_cta) {
  constexpr int kWarps = kUpdateThreads / 32;
  __shared__ ST red_s[32];
  __shared__ double sm_z[kWarps];
  __shared__ double sm_n[kUpdateMaxSteps][2][kWarps];
  __shared__ bool is_last;
  pdl_wait();   // launched as a programmatic dependent of the rollout kernel: its costs are read from here on
  const int t_first = blockIdx.x * steps_per_cta;
  const int n_t = min(steps_per_cta, p.T - t_first);
  const int k_chunk = (p.K + gridDim.y - 1) / gridDim.y;
  const int k_begin = blockIdx.y * k_chunk, k_end = min(p.K, k_begin + k_chunk);
  double* my_partial = partial ? partial + (size_t)blockIdx.y * (2 + 2 * p.T) : nullptr;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  // The kernel is a chain of memory round trips, so each thread fetches the costs AND the first step's controls of its
  // first kCached samples in one go and keeps them in registers across the min; the host cuts K into ranges of at most
  // kCached * blockDim samples, and anything beyond (a caller's single range) takes the two-pass route through L1.
  constexpr int kCached = kUpdateCached;
  ST sc[kCached];
  float2 uc[kCached];
  ST bmin = (ST)INFINITY;
#pragma unroll
  for (int j = 0; j < kCached; ++j) {
    const int k = k_begin + threadIdx.x + j * (int)blockDim.x;
    sc[j] = (ST)INFINITY;
    uc[j] = make_float2(0.0f, 0.0f);
    if (k < k_end) {
      RA_DEVICE_CHECK(k >= 0 && k < p.K && t_first < p.T);
      sc[j] = s_tilde_at<ST>(S_tilde, pen, k);
      uc[j] = __ldg(u + (long long)k * su_k + (long long)t_first * su_t);
    }
    bmin = min(bmin, sc[j]);
  }
  const int k_rest = k_begin + kCached * (int)blockDim.x;
  for (int k = k_rest + threadIdx.x; k < k_end; k += blockDim.x) bmin = min(bmin, s_tilde_at<ST>(S_tilde, pen, k));
  const ST beta = block_reduce<ST>(bmin, red_s, [](ST a, ST b) { return a < b ? a : b; }, (ST)INFINITY);

  // w~_k once per sample (an empty slot holds S~ = +inf, hence weight exactly 0), reused for every step of this CTA.
  // Z and the numerators are summed in fp64: with soft weights (ESS >> 1) and K = 65536 an fp32 sum would spend a
  // visible part of the 1e-4 budget of v+ on its own rounding.  Each w~ is an fp32 exp2 of an fp32 argument.
  float wc[kCached];
  double Z = 0.0;
#pragma unroll
  for (int j = 0; j < kCached; ++j) {
    wc[j] = exp2f((float)(sc[j] - beta) * p.neg_log2e_over_lambda);
    Z += (double)wc[j];
  }
  for (int k = k_rest + threadIdx.x; k < k_end; k += blockDim.x)
    Z += (double)exp2f((float)(s_tilde_at<ST>(S_tilde, pen, k) - beta) * p.neg_log2e_over_lambda);
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) Z += __shfl_xor_sync(0xFFFFFFFFu, Z, o);
  if (lane == 0) sm_z[warp] = Z;
  for (int tt = 0; tt < n_t; ++tt) {
    const int t = t_first + tt;
    float2 un[kCached];          // the next step's controls are fetched while this step's are summed
#pragma unroll
    for (int j = 0; j < kCached; ++j) {
      const int k = k_begin + threadIdx.x + j * (int)blockDim.x;
      un[j] = (tt + 1 < n_t && k < k_end) ? __ldg(u + (long long)k * su_k + (long long)(t + 1) * su_t) : make_float2(0.0f, 0.0f);
    }
    double n0 = 0.0, n1 = 0.0;
#pragma unroll
    for (int j = 0; j < kCached; ++j) {
      n0 = fma((double)wc[j], (double)uc[j].x, n0);
      n1 = fma((double)wc[j], (double)uc[j].y, n1);
      uc[j] = un[j];
    }
    for (int k = k_rest + threadIdx.x; k < k_end; k += blockDim.x) {
      const float w = exp2f((float)(s_tilde_at<ST>(S_tilde, pen, k) - beta) * p.neg_log2e_over_lambda);
      const float2 uk = __ldg(u + (long long)k * su_k + (long long)t * su_t);
      n0 = fma((double)w, (double)uk.x, n0);
      n1 = fma((double)w, (double)uk.y, n1);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {   // fixed-order tree inside the warp ...
      n0 += __shfl_xor_sync(0xFFFFFFFFu, n0, o);
      n1 += __shfl_xor_sync(0xFFFFFFFFu, n1, o);
    }
    if (lane == 0) { sm_n[tt][0][warp] = n0; sm_n[tt][1][warp] = n1; }
  }
  __syncthreads();
  // ... then over the warps, in order: thread (tt, i) finishes N_t[i]; every thread that needs Z forms the same sum
  double Zt = 0.0;
#pragma unroll
  for (int w = 0; w < kWarps; ++w) Zt += sm_z[w];
  const int my_tt = threadIdx.x >> 1, my_i = threadIdx.x & 1;
  double N = 0.0;
  if (my_tt < n_t) {
#pragma unroll
    for (int w = 0; w < kWarps; ++w) N += sm_n[my_tt][my_i][w];
  }
  // one range, no closed-loop tail: this CTA owns its v+_t outright, no exchange needed
  if (my_partial && done && gridDim.y == 1 && !tail.x0g) my_partial = nullptr;
  if (my_partial) {   // the range's / shard's unnormalised share {beta_g, Z_g, N_g[T][2]}
    RA_DEVICE_CHECK(my_tt >= n_t || (t_first + my_tt < p.T && n_t <= kUpdateMaxSteps));
    if (my_tt < n_t) my_partial[2 + 2 * (t_first + my_tt) + my_i] = N;
    if (threadIdx.x == 0 && blockIdx.x == 0) { my_partial[0] = (double)beta; my_partial[1] = Zt; }
    if (!done) return;
    // last CTA to finish combines: its ticket is the last one, so every other CTA's partials are in L2
    __syncthreads();             // this CTA's partial stores precede its ticket
    if (threadIdx.x == 0) {
      __threadfence();
      const unsigned int ticket = atomicAdd(done, 1u);
      is_last = ticket == gridDim.x * gridDim.y - 1u;
      if (is_last) *done = 0u;   // armed for the next launch
      __threadfence();
    }
    __syncthreads();
    if (!is_last) return;
    combine_partials_cta(p, partial, (int)gridDim.y, v_out);
    if (tail.x0g) {
      __syncthreads();           // v+ complete before it is applied and shifted
      plant_shift_any(p, tail.x0g, v_out, nullptr, tail.log, tail.loop);
    }
    return;
  }
  if (my_tt < n_t) v_out[2 * (t_first + my_tt) + my_i] = clampf((float)(N / Zt), p.u_min[my_i], p.u_max[my_i]);
  if (blockIdx.x == 0 && threadIdx.x == 0 && stats) { stats[0] = (float)beta; stats[1] = (float)Zt; }
  if (blockIdx.x == 0 && w_out) {
    const float invZ = (float)(1.0 / Zt);
    for (int k = threadIdx.x; k < p.K; k += blockDim.x)
      w_out[k] = exp2f((float)(s_tilde_at<ST>(S_tilde, pen, k) - beta) * p.neg_log2e_over_lambda) * invZ;
  }
}

// [T][K] scratch -> caller's [K][T][2] (diagnostic output of ra_mppi_rollout_costs)
__global__ void export_u_kernel(const __grid_constant__ Params p, float2* __restrict__ out) {
  const long long n = (long long)p.K * p.T;
  for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n;
       i += (long long)gridDim.x * blockDim.x) {
    const int k = (int)(i / p.T), t = (int)(i % p.T);
    out[i] = p.u_raw[(size_t)t * p.K + k];
  }
}

__global__ void export_costs_kernel(const __grid_constant__ Params p, float* __restrict__ S,
                                    float* __restrict__ cvar, float* __restrict__ S_tilde) {
  const int k = blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= p.K) return;
  if (S) S[k] = (float)p.S[k];
  if (cvar) cvar[k] = p.cvar[k];
  if (S_tilde) S_tilde[k] = (float)(p.S[k] + p.pen[k]);
}

// fp64 S and S~ = S + J_C of the context scratch (ra_mppi_export_costs_f64)
__global__ void export_costs_f64_kernel(const __grid_constant__ Params p, double* __restrict__ S,
                                        double* __restrict__ S_tilde) {
  const int k = blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= p.K) return;
  if (S) S[k] = p.S[k];
  if (S_tilde) S_tilde[k] = p.S[k] + p.pen[k];
}

// Parity hooks: raw Philox words and state-noise draws exactly as the rollout kernel makes them.
__global__ void philox_probe_kernel(const __grid_constant__ Params p, const uint4* __restrict__ ctr,
                                    int n, uint4* __restrict__ out) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) out[i] = philox4x32_10(ctr[i].x, ctr[i].y, ctr[i].z, ctr[i].w, p.rk);
}

template <int NX, int NOISE>
__global__ void noise_probe_kernel(const __grid_constant__ Params p, const int* __restrict__ kmt, int n,
                                   float* __restrict__ w) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  float z[NX];
  state_noise<NX, NOISE>(p, (uint32_t)kmt[3 * i], (uint32_t)kmt[3 * i + 1], (uint32_t)kmt[3 * i + 2],
                         iteration_field(p, STREAM_W), z);
#pragma unroll
  for (int j = 0; j < NX; ++j) w[(size_t)i * NX + j] = z[j] * p.wscale[j];
}

// Materialised-noise generator: w[K][T][NX][M_pad] = sigma_w (.) z, the same draws the fused
// kernel makes in registers (HBM-roofline mode of BASELINE.json).  A streaming kernel: consecutive threads take
// consecutive m, so every row of M_pad floats is written in full 128-byte lines.  Where a Philox call serves two
// steps (two words per step: n_x = 4, Gaussian or uniform) a thread owns one CALL and writes both steps' rows, so no
// call is computed twice and half discarded (round 2 did: one thread per (k, t, m) through state_noise).
template <int NX, int NOISE>
__global__ void __launch_bounds__(256) materialise_noise_kernel(const __grid_constant__ Params p,
                                                                float* __restrict__ w) {
  const uint32_t c3 = iteration_field(p, STREAM_W);
  const long long stride = (long long)gridDim.x * blockDim.x;
  const long long i0 = blockIdx.x * (long long)blockDim.x + threadIdx.x;
  const size_t step_floats = (size_t)NX * p.M_pad;
  if constexpr (NoiseWords<NX, NOISE>::value == 2) {
    const int TP = (p.T + 1) / 2;                      // Philox calls per realisation: steps (2 tp, 2 tp + 1)
    const long long n = (long long)p.K * TP * p.M_pad;
    for (long long i = i0; i < n; i += stride) {
      const int m = (int)(i % p.M_pad);
      const long long ktp = i / p.M_pad;
      const int tp = (int)(ktp % TP), k = (int)(ktp / TP), t = 2 * tp;
      const uint4 q = philox4x32_10((uint32_t)(k + p.k_off), (uint32_t)m, (uint32_t)tp, c3, p.rk);
      RA_DEVICE_CHECK(k < p.K && t < p.T && m < p.M_pad);
      float* o = w + ((size_t)k * p.T + t) * step_floats + m;
      float z[NX];
      const uint32_t w0[2] = {q.x, q.y};
      noise_from_words<NX, NOISE>(p, w0, z);
#pragma unroll
      for (int j = 0; j < NX; ++j) __stcs(o + (size_t)j * p.M_pad, z[j] * p.wscale[j]);
      if (t + 1 < p.T) {                               // an odd horizon ends on the first half of its last call
        const uint32_t w1[2] = {q.z, q.w};
        noise_from_words<NX, NOISE>(p, w1, z);
        o += step_floats;
#pragma unroll
        for (int j = 0; j < NX; ++j) __stcs(o + (size_t)j * p.M_pad, z[j] * p.wscale[j]);
      }
    }
  } else {
    const long long n = (long long)p.K * p.T * p.M_pad;
    for (long long i = i0; i < n; i += stride) {
      const int m = (int)(i % p.M_pad);
      const long long kt = i / p.M_pad;
      const int t = (int)(kt % p.T), k = (int)(kt / p.T);
      float z[NX];
      state_noise<NX, NOISE>(p, (uint32_t)(k + p.k_off), (uint32_t)m, (uint32_t)t, c3, z);
      float* o = w + (size_t)kt * step_floats + m;
#pragma unroll
      for (int j = 0; j < NX; ++j) o[(size_t)j * p.M_pad] = z[j] * p.wscale[j];
    }
  }
}

}  // namespace ra
