/*
 * RA-MPPI ORACLE — TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, single-threaded-by-definition fp64 CPU implementation of one
 * Risk-Aware MPPI controller iteration, written step by step from the paper
 * (arXiv 2209.12842; citations are PAPER.md line numbers + equation/algorithm).
 * It shares no code, header, table or constant with the CUDA path under
 * paper_2209_12842_b200/.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may call it.
 *
 * Notation: the BASELINE letters are used (K control samples = paper's M,
 * M noise realisations per sample = paper's N, T horizon steps = paper's K).
 *
 * Pins (tests/test_oracle_*.py, all `-m "not gpu"`):
 *   philox4x32_10        - agreement with ATen's at::philox_engine (compiled from
 *                          torch's header by the test) and cuRAND's host generator
 *   box_muller           - moments of 2^19 draws, exact end points
 *   box_muller16         - exact end points, exact lattice moments, sample moments, Kolmogorov-Smirnov
 *                          distance and tail mass at the alpha quantiles in use, word / half-word layout
 *   cvar_topk / literal  - brute force on hand arrays, Rockafellar-Uryasev
 *                          identity, closed-form Gaussian CVaR
 *   dynamics             - closed-form Euler sums, straight-line / steady-state
 *                          single-track, Euler order check against a separate RK4
 *   costs                - hand-computed points, bilinear reproduces affine maps
 *   weights/update       - sum to 1, shift invariance, lambda limits
 *   control draw (O1a)   - std(u - v) = sigma_eps per component (distinct sigmas), mean 0,
 *                          uncorrelated; u = v + sigma_eps (.) box_muller(r0, r1) of the EPS
 *                          counter bit for bit through the free functions above
 *   iteration end-to-end - Gaussian closed-form CVaR through the whole rollout
 *                          path with the test-only linear risk; sigma_w=0, A=0,
 *                          M=1, K=1 special cases
 * "parity unpinned" (defined by BASELINE.json configs, not by the paper): the
 * numeric constants of the vehicle models and the cost weights of the configs.
 */
#ifndef RA_MPPI_ORACLE_H
#define RA_MPPI_ORACLE_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

enum { ORC_DYN_BICYCLE = 0, ORC_DYN_SINGLE_TRACK = 1 };
enum { ORC_NOM_GOAL = 0, ORC_NOM_ELLIPSE_TRACK = 1, ORC_NOM_RACING = 2 };
enum { ORC_RISK_CIRCLES = 0, ORC_RISK_COSTMAP = 1, ORC_RISK_LINEAR_STATE = 2, ORC_RISK_NOMINAL = 3 /* l = q */ };
enum { ORC_NOISE_GAUSSIAN = 0, ORC_NOISE_UNIFORM = 1, ORC_NOISE_JUMP = 2 };
enum { ORC_STREAM_EPS = 0, ORC_STREAM_W = 1, ORC_STREAM_PLANT = 2 };

typedef struct {
  int32_t K, M, T;          /* samples, realisations, horizon                          */
  double  dt;
  int32_t dyn;              /* ORC_DYN_*                                               */
  double  dyn_p[8];         /* bicycle {L}; single-track {m,Iz,lf,lr,Cf,Cr,vx_floor}   */
  double  u_min[2], u_max[2];
  double  sigma_eps[2];     /* sqrt(diag Sigma_eps), (2c) PAPER.md:42                  */
  double  sigma_w[6];       /* additive per-step state noise scale, (6) PAPER.md:63    */
  double  alpha, lambda, gamma;     /* (8b) :81, (5)/(17) :55/:134, (3) :47            */
  double  A, B, C_u, eta;           /* (14) :120, (18) :144, (15) :124, Alg.1 l.7 :183 */
  int32_t nominal;          /* ORC_NOM_*                                               */
  double  nom_p[12];        /* goal {w,gx,gy,w_phi}; track {a,b,half_w,w_lat,w_v,v_ref,w_bdry,w_phi};
                               racing {ax,ay,rc,half_w,c1,c2,c3,c4,c5} (20)-(23) PAPER.md:164-241 */
  int32_t risk;             /* ORC_RISK_*                                              */
  double  risk_p[4];        /* circles {weight,margin}; costmap {weight}; linear {weight,index} */
  int32_t noise_kind;       /* ORC_NOISE_*                                             */
  double  noise_p[4];       /* uniform: unused (half-width = sigma_w); jump {prob}, magnitude = sigma_w */
  uint64_t seed;
  /* environment (borrowed pointers) */
  const double* circles;  int32_t n_circles;        /* [n,3] x,y,r                     */
  const double* costmap;  int32_t map_h, map_w;     /* row-major [h][w]                */
  double  map_res, map_ox, map_oy;
} orc_problem;

/* ---- random source ---------------------------------------------------- */
void   orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]);
void   orc_counter(uint32_t k, uint32_t m, uint32_t t, uint32_t J, uint32_t j,
                   uint32_t stream, uint64_t iteration, uint32_t ctr[4]);
void   orc_box_muller(uint32_t ra, uint32_t rb, double z[2]);   /* 23-bit uniforms, two words (control draw eps) */
void   orc_box_muller16(uint32_t w, double z[2]);                /* one word: 16-bit radius, 23-bit angle (state noise) */
/* the n_x noise values added to the state at step t of realisation (k,m)     */
void   orc_state_noise(const orc_problem* p, uint32_t k, uint32_t m, uint32_t t,
                       uint32_t stream, uint64_t iteration, double w[6]);

/* ---- models ------------------------------------------------------------ */
int    orc_nx(int32_t dyn);
void   orc_dynamics(const orc_problem* p, const double* x, const double u[2], double* x_next);
double orc_q(const orc_problem* p, const double* x);     /* nominal running cost */
double orc_phi(const orc_problem* p, const double* x, const double* x0);   /* terminal cost (x0: racing progress) */
double orc_l(const orc_problem* p, const double* x);     /* risk running cost    */
double orc_ellipse_offset(double a, double b, double X, double Y);
double orc_bilinear(const orc_problem* p, double X, double Y);
/* rounded-rectangle race track: lateral deviation e (+ outward) and centreline arc length s  */
double orc_racing_offset(const orc_problem* p, double X, double Y);
double orc_racing_arclength(const orc_problem* p, double X, double Y);
/* smallest |d_i - r_i| over the obstacles at (X,Y): distance of the indicator (22) from its jump */
double orc_indicator_margin(const orc_problem* p, double X, double Y);
/* smallest |d_i - (r_i + margin)|: distance of the hinge risk cost from its switch between exactly 0 and > 0 */
double orc_hinge_margin(const orc_problem* p, double X, double Y);

/* ---- CVaR -------------------------------------------------------------- */
int32_t orc_tail_count(double alpha, int32_t M);
double  orc_cvar_topk(const double* L, int32_t M, int32_t k_tail);
double  orc_cvar_literal12(const double* L, int32_t M, double alpha);
void    orc_sensitivity_scale(const double* L, int32_t M, double B, double* La);

/* ---- one controller iteration ------------------------------------------ */
/* O1 for samples k in [k_begin,k_end): all outputs indexed by (k-k_begin).
 * Any output pointer may be NULL.  n_threads>1 splits the k range over
 * std::threads (results identical: every k is independent).                */
int orc_rollout_costs(const orc_problem* p, const double* x0, const double* v,
                      uint64_t iteration, int32_t k_begin, int32_t k_end, int32_t n_threads,
                      double* u /*[n,T,2]*/, double* S /*[n]*/, double* cvar /*[n]*/,
                      double* S_tilde /*[n]*/, double* L /*[n,M]*/, double* xT /*[n,M,nx]*/,
                      double* x_nom /*[n,nx] nominal terminal state*/,
                      double* margin /*[n,M+1] min over t of the indicator margin (racing costs; col 0 nominal, 1..M noisy)
                                        or of the hinge margin (circle risk; cols 1..M, col 0 = inf); or NULL*/);
/* O2-O3: weights and update from S_tilde[K] and u[K,T,2].                   */
int orc_weights_update(const orc_problem* p, const double* S_tilde, const double* u,
                       double* v_plus /*[T,2]*/, double* w /*[K]*/, double* Z, double* beta);
/* O0-O3: full iteration.                                                    */
int orc_step(const orc_problem* p, const double* x0, const double* v, uint64_t iteration,
             int32_t n_threads, double* v_plus /*[T,2]*/);
/* closed-loop glue (BASELINE config 4): plant and warm-start shift.         */
void orc_plant_step(const orc_problem* p, const double* x0, const double u0[2],
                    uint64_t iteration, double* x_next);
void orc_shift(const double* v_plus, int32_t T, double* v_next);

#ifdef __cplusplus
}
#endif
#endif
