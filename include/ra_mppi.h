/*
 * ra_mppi.h — C ABI of the B200-native RA-MPPI hot path (arXiv 2209.12842).
 *
 * One controller iteration of Risk-Aware MPPI (Algorithm 1, :167-223;
 * Fig. 1 :74) as hand-written sm_100a CUDA kernels.  Letters follow BASELINE.json:
 * K control samples (paper's M), M noise realisations per sample (paper's N),
 * T horizon steps (paper's K).
 *
 * Conventions for every entry point
 *  - Pointers named d_* are DEVICE pointers on the context's device; all other
 *    pointers are HOST pointers.  Row-major, fp32 unless stated.
 *  - ra_mppi_step / ra_mppi_rollout_costs / ra_mppi_plant_shift only enqueue work on
 *    `cuda_stream` (a cudaStream_t passed as void*; NULL = legacy default stream).
 *    They do not synchronise, allocate or free, so they can be captured in a graph.
 *  - The context owns its scratch (copies of the environment, u[T,K], S, CVaR, S~,
 *    optional materialised noise).  The caller owns every pointer it passes; the
 *    library keeps none of them past the enqueued work.
 *  - Errors are returned as ra_status; nothing throws, nothing calls exit().
 *    There is no CPU fallback: without an sm_100 device ra_mppi_create fails.
 *  - One context per stream; not re-entrant.
 *  - Every entry point makes the context's device current for its own duration and restores the
 *    caller's current device before returning.
 */
#ifndef RA_MPPI_H
#define RA_MPPI_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct ra_mppi_ctx ra_mppi_ctx; /* opaque */

typedef enum {
  RA_OK = 0,
  RA_EINVAL = 1,       /* null pointer, size <= 0, parameter out of its domain, struct_size mismatch */
  RA_EUNSUPPORTED = 2, /* M or T outside the supported set, device is not sm_100 */
  RA_ECUDA = 3,        /* a CUDA call failed (see ra_mppi_last_error) */
  RA_ENOMEM = 4        /* device allocation failed */
} ra_status;

typedef enum { RA_DYN_KINEMATIC_BICYCLE = 0, RA_DYN_SINGLE_TRACK = 1 } ra_dyn;
typedef enum { RA_NOM_GOAL = 0, RA_NOM_ELLIPSE_TRACK = 1, RA_NOM_RACING = 2 /* (20)-(23) PAPER.md:164-241 */ } ra_nominal;
typedef enum {
  RA_RISK_CIRCLES = 0, RA_RISK_COSTMAP = 1, RA_RISK_LINEAR_STATE = 2 /* test-only */,
  RA_RISK_NOMINAL = 3 /* l = q; with RA_NOM_RACING */
} ra_risk;
typedef enum { RA_NOISE_GAUSSIAN = 0, RA_NOISE_UNIFORM = 1, RA_NOISE_JUMP = 2 } ra_noise_kind;
typedef enum { RA_NOISE_FUSED = 0, RA_NOISE_MATERIALISED = 1 } ra_noise_mode;

#define RA_MAX_M 512 /* realisations per sample: 1..RA_MAX_M                                  */
#define RA_MAX_T 128 /* horizon steps: 1..RA_MAX_T                                            */

/* Problem statement (8a)-(8c) PAPER.md:78-85 and Algorithm 1 "Given" :170. */
typedef struct {
  uint32_t struct_size; /* = sizeof(ra_mppi_config)                                           */
  int32_t K, M, T;      /* samples, realisations, horizon (PAPER.md:247 gives 1024, 300, 30)   */
  float dt;             /* Euler step of F (1) PAPER.md:29                                    */
  int32_t dyn;          /* ra_dyn                                                             */
  float dyn_p[8];       /* bicycle {wheelbase}; single-track {m,Iz,lf,lr,Cf,Cr,vx_floor}      */
  float u_min[2], u_max[2]; /* control clamps, applied inside F and to v+                     */
  float sigma_eps[2];   /* sqrt(diag Sigma_eps), control sampling noise (2c) PAPER.md:42      */
  float sigma_w[6];     /* per-step additive state noise scale, w_k of (6) PAPER.md:63        */
  float alpha;          /* CVaR confidence level in (0,1), (8b) PAPER.md:81-87                */
  float lambda;         /* temperature of (5)/(17) PAPER.md:55,:134; > 0                      */
  float gamma;          /* control-cost weight of (3) PAPER.md:47-49; >= 0                    */
  float A;              /* CVaR penalty weight (14) PAPER.md:120                              */
  float B;              /* risk sensitivity scale (18) PAPER.md:144; > 0                      */
  float C_u;            /* CVaR bound (8b)/(15) PAPER.md:81,:124                              */
  float eta;            /* fraction of zero-mean samples, Alg.1 l.7 PAPER.md:183,:247; [0,1)  */
  int32_t nominal;      /* ra_nominal: q(x), phi(x) of (3)                                    */
  float nom_p[12];      /* goal {w,gx,gy,w_phi}; track {a,b,half_w,w_lat,w_v,v_ref,w_bdry,w_phi};
                           racing {ax,ay,rc,half_w,c1,c2,c3,c4,c5}: rounded-rectangle track, costs (20)-(23) */
  int32_t risk;         /* ra_risk: l(x~) of (9) PAPER.md:93                                  */
  float risk_p[4];      /* circles {weight,margin}; costmap {weight}; linear {weight,index}   */
  int32_t noise_kind;   /* ra_noise_kind                                       */
  float noise_p[4];     /* jump {probability}; otherwise unused                               */
  int32_t noise_mode;   /* ra_noise_mode: fused = Philox in registers; materialised = w[K,T,M,nx] in HBM */
  uint64_t seed;        /* Philox4x32-10 key                                                  */
  int32_t device;       /* CUDA device ordinal                                                */
  /* K-sharding over several contexts / GPUs (not in the paper): this context
   * holds the K samples with global indices k_offset .. k_offset+K-1 of K_total.  Philox counters and
   * the eta split (Alg.1 l.7) use the global index, so results do not depend on the partition.
   * K_total = 0 means "not sharded" (K_total = K, k_offset must be 0).                             */
  int32_t k_offset;
  int32_t K_total;
} ra_mppi_config;

/* Environment; HOST pointers, copied at create (caller keeps ownership). */
typedef struct {
  const float* circles; /* [n_circles,3] x,y,r (obstacle set)                */
  int32_t n_circles;
  const float* costmap; /* [map_h][map_w] row-major; cell (iy,ix) centre = origin + (i+0.5)*res */
  int32_t map_h, map_w;
  float map_res, map_ox, map_oy;
} ra_mppi_env;

/* Allocate a controller context on cfg->device.  cfg/env: host.  *out receives the
 * context (NULL on failure).  RA_EINVAL / RA_EUNSUPPORTED / RA_ECUDA / RA_ENOMEM.        */
ra_status ra_mppi_create(const ra_mppi_config* cfg, const ra_mppi_env* env, ra_mppi_ctx** out);
/* Why the calling thread's most recent ra_mppi_create failed ("" after a success): there is no context yet whose
 * ra_mppi_last_error could say it.  Owned by the library, valid until this thread's next create call.            */
const char* ra_mppi_create_error(void);

/* Replace the environment of an existing context (moving obstacles, a refreshed costmap): env is HOST memory,
 * copied before the call returns.  Up to 1024 circles; a costmap must keep the map_h x map_w it had at create
 * (resolution and origin may change).  Synchronises the device and drops the captured closed-loop graph.
 * Not capturable.  RA_EINVAL / RA_EUNSUPPORTED / RA_ECUDA.                                                */
ra_status ra_mppi_set_env(ra_mppi_ctx* ctx, const ra_mppi_env* env);

/* One full iteration, Alg.1 l.3-31: sample u^k = v + eps^k, nominal
 * and noisy rollouts, risk costs (9), CVaR (12), soft filter (14)-(16), weights (17),
 * update (4).  d_x0 [n_x] current state; d_v [T,2] in: mean control v, out: v+ (clamped).
 * `iteration` enters the Philox counter (low 28 bits).                                    */
ra_status ra_mppi_step(ra_mppi_ctx* ctx, const float* d_x0, float* d_v, uint64_t iteration,
                       void* cuda_stream);

/* The same iteration stopped after Alg.1 l.29: per-sample costs.  Outputs (device, any may
 * be NULL): d_S [K] nominal cost (3); d_cvar [K] CVaR_alpha of the (scaled) risk costs;
 * d_S_tilde [K] modified cost (16); d_L [K,M] raw risk costs (9); d_xT [K,M,n_x] final
 * noisy states; d_u [K,T,2] sampled controls u^k (unclamped).  d_v is not modified.       */
ra_status ra_mppi_rollout_costs(ra_mppi_ctx* ctx, const float* d_x0, const float* d_v,
                                uint64_t iteration, float* d_S, float* d_cvar, float* d_S_tilde,
                                float* d_L, float* d_xT, float* d_u, void* cuda_stream);

/* K-sharded iteration, local part: Alg.1 l.3-29 on this context's samples, then the shard's share of
 * (17)/(4): d_partial [2+2T] fp64 (device) = { beta_g = min_k S~_k, Z_g = sum_k exp(-(S~_k-beta_g)/lambda),
 * N_g[T][2] = sum_k exp(-(S~_k-beta_g)/lambda) u^k_t } over the local k.  d_v is read only.           */
ra_status ra_mppi_step_partial(ra_mppi_ctx* ctx, const float* d_x0, const float* d_v, uint64_t iteration,
                               double* d_partial, void* cuda_stream);
/* K-sharded iteration, exchange step: d_partials [n_parts][2+2T] fp64 (device; the shards' partials,
 * e.g. after an NCCL all-gather, any order) -> d_v_plus [T,2] = clamp(sum_g s_g N_g / sum_g s_g Z_g),
 * s_g = exp(-(beta_g - min_g beta_g)/lambda): exactly (17)/(4) over the union of the shards.        */
ra_status ra_mppi_combine_partials(ra_mppi_ctx* ctx, const double* d_partials, int32_t n_parts,
                                   float* d_v_plus, void* cuda_stream);

/* The fp64 cost scratch of the most recent step / rollout_costs on this context: d_S64 [K],
 * d_S_tilde64 [K] (device, fp64, either may be NULL).  The weights (17) are formed from these
 * fp64 values; the fp32 outputs of ra_mppi_rollout_costs are their roundings.               */
ra_status ra_mppi_export_costs_f64(ra_mppi_ctx* ctx, double* d_S64, double* d_S_tilde64, void* cuda_stream);

/* Weights (17)/(5) and update (4) alone, from caller-supplied costs and controls:
 * d_S_tilde [K], d_u [K,T,2] -> d_v_plus [T,2] (clamped), d_w [K] normalised weights or
 * NULL, d_stats [2] = {beta~, Z} or NULL.                                                 */
ra_status ra_mppi_weights_update(ra_mppi_ctx* ctx, const float* d_S_tilde, const float* d_u,
                                 float* d_v_plus, float* d_w, float* d_stats, void* cuda_stream);

/* Weights (17) PAPER.md:134 and update (4) PAPER.md:51 for callers that must not allocate device memory.
 *
 * Who this is for: code that runs where cudaMalloc is off limits -- a control loop that has already handed all of
 * its device memory to a fixed pool, a plug-in loaded into a host process whose allocator it may not touch, a
 * real-time thread in which an allocation (an implicit device synchronisation and an unbounded driver call) would
 * break the deadline.  Such a caller cannot use a context either, because creating one allocates.  This call needs
 * no context and calls no cudaMalloc, cudaFree or allocating library routine: the per-range partial sums and the
 * ticket counter that the multi-range weights/update kernel exchanges through global memory live in a fixed array
 * of RA_STATIC_SCRATCH_BYTES bytes compiled into the library.  Every GPU that loads the library holds that array
 * until the process exits, used or not; that is the price, and why the limits below are modest.
 *
 *   K in 1..RA_STATIC_MAX_K samples, T in 1..RA_MAX_T steps, lambda > 0; u_min[2], u_max[2] HOST (the clamp of v+);
 *   d_S_tilde [K] modified costs (16), d_u [K,T,2] sampled controls, d_v_plus [T,2] output: DEVICE pointers on the
 *   CURRENT device (there is no context to name one).  Same arithmetic as the context's weights/update kernel
 *   (fp32 exp2, fp64 sums, fixed summation order): results are reproducible run to run, and agree with the
 *   context-based weights/update call to rounding (the samples are summed range by range instead of in one pass).
 *
 * Sizes beyond the limits are refused with RA_EUNSUPPORTED before anything is enqueued; RA_EINVAL for a null pointer,
 * K or T < 1, a non-positive or non-finite lambda, u_min > u_max; RA_ECUDA when a CUDA call fails.  The reason is kept
 * per calling thread and read with ra_mppi_weights_update_static_error.
 *
 * The first call on each device looks up the device address of the array (the array's name is only a host-side
 * handle; kernels need the address the runtime reports for the device that is current) and the SM count.  That
 * first call may make the runtime load the library's code onto the device, so make it once at start-up, outside
 * any stream capture.  Later calls only enqueue a 4-byte memset (the ticket counter must start at zero whatever an
 * earlier, possibly aborted, call left behind) and one kernel on `cuda_stream`, and do not synchronise.
 *
 * All calls on a device share the one array.  Two calls whose kernels can overlap on the GPU (different streams
 * without an ordering between them, or two host threads) race on it and give wrong results: order them on one
 * stream or with events.  The array keeps the previous call's partial sums; every entry a call reads it has first
 * written itself, so nothing but the ticket needs clearing.                                                    */
#define RA_STATIC_MAX_K 131072      /* 64 sample ranges of 2048                                               */
#define RA_STATIC_SCRATCH_BYTES 132352 /* 64 x (2 + 2 x RA_MAX_T) fp64 partial sums + a 256-byte ticket slot    */
ra_status ra_mppi_weights_update_static(int32_t K, int32_t T, float lambda, const float* u_min, const float* u_max,
                                        const float* d_S_tilde, const float* d_u, float* d_v_plus,
                                        void* cuda_stream);
/* Why the calling thread's most recent ra_mppi_weights_update_static call failed ("" if it did not).  The text is
 * owned by the library and valid until this thread's next call of that function.                                */
const char* ra_mppi_weights_update_static_error(void);

/* Closed-loop glue, Alg.1 l.32-33 on a simulated plant (BASELINE config 4):
 * d_x0 <- F~(d_x0, v+_0, w_plant(iteration)); d_u_applied [2] <- v+_0 (or NULL);
 * d_v[t] <- d_v[t+1], d_v[T-1] kept (warm-start shift).                                   */
ra_status ra_mppi_plant_shift(ra_mppi_ctx* ctx, float* d_x0, float* d_v, float* d_u_applied,
                              uint64_t iteration, void* cuda_stream);

/* n_iter receding-horizon iterations (step + plant_shift) replayed from one captured CUDA
 * graph with a device-resident iteration counter starting at `iteration0`.  d_log
 * [n_iter, n_x+2] receives (state after the plant step, applied control) per iteration, or
 * NULL.  h_ms [n_iter] (HOST) receives per-iteration device milliseconds (CUDA events) or
 * NULL; when non-NULL the call synchronises the stream before returning.                  */
ra_status ra_mppi_closed_loop(ra_mppi_ctx* ctx, float* d_x0, float* d_v, uint64_t iteration0,
                              int32_t n_iter, float* d_log, float* h_ms, void* cuda_stream);

/* ra_mppi_step with HOST buffers: h_x0 [n_x] and h_v [T,2] (in: v, out: v+) go through the context's pinned
 * staging buffer (one host-to-device copy of iteration, x0 and v together, the step, one device-to-host copy of v+),
 * submitted as one CUDA graph captured on first use; the call returns after the stream has drained with v+ in h_v.
 * Any host memory works (pinned or pageable).  Results are bit-identical to ra_mppi_step on device buffers.       */
ra_status ra_mppi_step_host(ra_mppi_ctx* ctx, const float* h_x0, float* h_v, uint64_t iteration,
                            void* cuda_stream);

/* Kernel timing for roofline accounting: when enabled, every step / rollout_costs records a CUDA
 * event pair around the fused rollout kernel on the launching stream.
 * ra_mppi_last_rollout_ms waits for that pair and returns its milliseconds in *h_ms (HOST); RA_EINVAL when
 * no rollout kernel has been timed (timing never enabled, only A = 0 steps, or only graph-captured steps).   */
ra_status ra_mppi_enable_kernel_timing(ra_mppi_ctx* ctx, int32_t enable);
ra_status ra_mppi_last_rollout_ms(ra_mppi_ctx* ctx, float* h_ms);

/* Raw generator access for parity tests: out[n,4] = Philox4x32-10(ctr[n,4], key(seed)).   */
ra_status ra_mppi_philox(ra_mppi_ctx* ctx, const uint32_t* d_ctr, int32_t n, uint32_t* d_out,
                         void* cuda_stream);
/* State-noise draws exactly as the rollout kernel makes them: d_w [n, n_x] for the n
 * triples d_kmt [n,3] = (k, m, t) of stream W at `iteration`.                             */
ra_status ra_mppi_state_noise(ra_mppi_ctx* ctx, const int32_t* d_kmt, int32_t n,
                              uint64_t iteration, float* d_w, void* cuda_stream);

/* Measured issue rates of the plain SM pipes on `device`, in 1e12 lane-operations per second:
 * h_tera_lane_ops[4] (HOST) = {FFMA, IMAD.WIDE.U32 each paired with one LOP3 (the Philox round
 * pattern), LOP3, MUFU.LG2}.  Runs four short
 * microbenchmark kernels on the NULL stream and synchronises.  Roofline denominators only.   */
ra_status ra_mppi_measure_pipe_peaks(int32_t device, float* h_tera_lane_ops);

/* The two integer decisions ra_mppi_create derives from fp32 parameters, without touching a device (host only):
 * *h_k_tail = ceil((1-alpha) M) clamped to [1, M], the CVaR tail size of Alg.1 l.25-26 ((12) :107);
 * *h_K0 = ceil((1-eta) K_total), the number of samples that carry the mean control (Alg.1 l.7-10).
 * alpha and eta arrive as fp32, so both counts are taken with a guard of 2^-23 n against their representation
 * error (alpha = 0.7f with M = 10 counts 3, eta = 0.7f with K = 1000 counts 300).  Either pointer may be NULL.
 * RA_EINVAL: null cfg, struct_size mismatch, M or K <= 0, alpha outside (0,1), eta outside [0,1).            */
ra_status ra_mppi_query_counts(const ra_mppi_config* cfg, int32_t* h_k_tail, int32_t* h_K0);

/* Which instantiation of the rollout kernel this context launches (host only): h_variant[5] (HOST) =
 * {dynamics, risk, noise variant (ra_noise_kind, or 3 = materialised), realisation slots per lane, 1 if half a warp
 * carries a sample (M <= 16) else 0} -- the template arguments noisy_rollout_kernel<...> shows in a profiler, so that a
 * stored profiler capture can be matched against the kernel that is actually running.                              */
ra_status ra_mppi_rollout_variant(const ra_mppi_ctx* ctx, int32_t* h_variant);

/* Number of kernels one ra_mppi_step launches (for launch accounting).                   */
int32_t ra_mppi_launches_per_step(const ra_mppi_ctx* ctx);
/* Last error text, owned by the context (valid until the next call on it).               */
const char* ra_mppi_last_error(const ra_mppi_ctx* ctx);
/* Free everything the context owns.  NULL is a no-op.                                    */
ra_status ra_mppi_destroy(ra_mppi_ctx* ctx);

#ifdef __cplusplus
}
#endif
#endif /* RA_MPPI_H */
