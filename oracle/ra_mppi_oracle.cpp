/*
 * RA-MPPI ORACLE — TEST INFRASTRUCTURE, NOT THE PRODUCT (see ra_mppi_oracle.h).
 *
 * Plain fp64, one loop per index of the paper, no blocking / fusion / reordering.
 * Every function cites the PAPER.md passage it follows ("P:line").  Where the
 * paper is silent the reading is the one listed in DESIGN.md ("D:Gnn").
 *
 * parity unpinned (no paper value exists): vehicle-model constants and cost
 * weights, which come from BASELINE.json's configs.
 */
#include "ra_mppi_oracle.h"

#include <algorithm>
#include <cmath>
#include <cstring>
#include <functional>
#include <limits>
#include <thread>
#include <vector>

namespace {

const double kPi = 3.14159265358979323846264338327950288;

/* ---------------------------------------------------------------------------
 * Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11).  BASELINE.json fixes this
 * generator; the paper itself only says eps ~ N(0,Sigma_eps) (2c) P:42.
 * One round:  (hi0,lo0) = 0xD2511F53 * c0 ; (hi1,lo1) = 0xCD9E8D57 * c2
 *             c <- (hi1^c1^k0, lo1, hi0^c3^k1, lo0)
 * Between rounds the key is bumped by the Weyl constants.
 * ------------------------------------------------------------------------- */
inline void philox_round(uint32_t c[4], const uint32_t k[2]) {
  const uint64_t p0 = (uint64_t)0xD2511F53u * (uint64_t)c[0];
  const uint64_t p1 = (uint64_t)0xCD9E8D57u * (uint64_t)c[2];
  const uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
  const uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
  const uint32_t n0 = hi1 ^ c[1] ^ k[0];
  const uint32_t n1 = lo1;
  const uint32_t n2 = hi0 ^ c[3] ^ k[1];
  const uint32_t n3 = lo0;
  c[0] = n0; c[1] = n1; c[2] = n2; c[3] = n3;
}

inline double clampd(double x, double lo, double hi) { return x < lo ? lo : (x > hi ? hi : x); }

/* Number of 32-bit words one state step takes from the (k, m, stream, iteration) word stream.  State noise spends
 * 16 bits per uniform (D:RNG layout): one word carries one Box-Muller pair (two state components) or two uniform
 * draws, so a step takes n_x / 2 words, plus (jump noise) one word whose high half is the trigger. */
inline uint32_t words_per_step(const orc_problem* p) {
  const uint32_t nx = (uint32_t)orc_nx(p->dyn);
  return p->noise_kind == ORC_NOISE_JUMP ? nx / 2u + 1u : nx / 2u;
}

}  // namespace

extern "C" {

void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
  uint32_t c[4] = {ctr[0], ctr[1], ctr[2], ctr[3]};
  uint32_t k[2] = {key[0], key[1]};
  for (int r = 0; r < 10; ++r) {
    if (r > 0) { k[0] += 0x9E3779B9u; k[1] += 0xBB67AE85u; }
    philox_round(c, k);
  }
  out[0] = c[0]; out[1] = c[1]; out[2] = c[2]; out[3] = c[3];
}

/* D:RNG layout.  ctr = (k, m, t*J + j, stream<<28 | iteration&0x0FFFFFFF); the EPS stream uses J = 1, j = 0, and
 * the state-noise word stream passes its call index as t. */
void orc_counter(uint32_t k, uint32_t m, uint32_t t, uint32_t J, uint32_t j,
                 uint32_t stream, uint64_t iteration, uint32_t ctr[4]) {
  ctr[0] = k;
  ctr[1] = m;
  ctr[2] = t * J + j;
  ctr[3] = (stream << 28) | (uint32_t)(iteration & 0x0FFFFFFFull);
}

/* Box-Muller on two 23-bit uniforms (exactly representable in fp32 and fp64):
 * u1 = ((ra>>9)+1) 2^-23 in (0,1],  u2 = (rb>>9) 2^-23 in [0,1).  D:RNG layout. */
void orc_box_muller(uint32_t ra, uint32_t rb, double z[2]) {
  const double u1 = (double)((ra >> 9) + 1u) * (1.0 / 8388608.0);
  const double u2 = (double)(rb >> 9) * (1.0 / 8388608.0);
  const double rho = std::sqrt(-2.0 * std::log(u1));
  z[0] = rho * std::cos(2.0 * kPi * u2);
  z[1] = rho * std::sin(2.0 * kPi * u2);
}

/* Box-Muller pair from ONE Philox word (state-noise streams; D:RNG layout):
 * radius uniform  u1 = ((w & 0xFFFF) + 1/2) 2^-16 in (0,1)   (the low half of the word),
 * angle uniform   u2 = (w >> 9) 2^-23 in [0,1)               (the top 23 bits of the word),
 * both exactly representable in fp32 and fp64.  The two fields share bits 9..15 (the top 7 bits of u1 are the
 * bottom 7 bits of u2): for every radius the 2^16 remaining angles are equally spaced over the full turn, so the
 * pair has exactly the mixed moments of (radius lattice) x (uniform angle) and the 2^32 words still map to 2^32
 * distinct points.  |z| <= sqrt(2 * 17 ln 2) = 4.855 (truncated mass 1.2e-6 per draw); E z^2 = 1 - 5.3e-6,
 * E z^4 = 3 - 2.1e-4 on this lattice (exact sums, pinned in tests/test_oracle_rng.py). */
void orc_box_muller16(uint32_t w, double z[2]) {
  const double u1 = ((double)(w & 0xFFFFu) + 0.5) * (1.0 / 65536.0);
  const double u2 = (double)(w >> 9) * (1.0 / 8388608.0);
  const double rho = std::sqrt(-2.0 * std::log(u1));
  z[0] = rho * std::cos(2.0 * kPi * u2);
  z[1] = rho * std::sin(2.0 * kPi * u2);
}

int orc_nx(int32_t dyn) { return dyn == ORC_DYN_SINGLE_TRACK ? 6 : 4; }

/* w_t of (6) P:63 for realisation (k,m) at step t.  BASELINE configs: additive,
 * per step, not scaled by dt (D:G14).  Gaussian: sigma_w (.) N(0,I).  The two
 * non-Gaussian kinds are the paper's robustness experiment P:263:
 * uniform on [-sigma_w, sigma_w]; jump: with probability noise_p[0] a step of
 * length sigma_w (per-axis scale) in a uniformly random direction. */
void orc_state_noise(const orc_problem* p, uint32_t k, uint32_t m, uint32_t t,
                     uint32_t stream, uint64_t iteration, double w[6]) {
  const uint32_t nx = (uint32_t)orc_nx(p->dyn);
  const uint32_t Wd = words_per_step(p);
  const uint32_t key[2] = {(uint32_t)(p->seed & 0xFFFFFFFFull), (uint32_t)(p->seed >> 32)};
  /* D:RNG layout: the realisation (k, m) of a stream owns the word stream
   *   word n = output (n mod 4) of Philox4x32-10 at counter (k, m, n div 4, stream<<28 | iteration),
   * and step t takes the words Wd*t .. Wd*t + Wd - 1: word j carries state components 2j, 2j+1. */
  const uint32_t n0 = Wd * t, c_first = n0 / 4u, c_last = (n0 + Wd - 1u) / 4u;   /* at most 2 calls */
  uint32_t call[2][4];
  for (uint32_t c = c_first; c <= c_last; ++c) {
    uint32_t ctr[4];
    orc_counter(k, m, c, 1u, 0u, stream, iteration, ctr);
    orc_philox4x32_10(ctr, key, call[c - c_first]);
  }
  uint32_t r[4];
  for (uint32_t i = 0; i < Wd; ++i) r[i] = call[(n0 + i) / 4u - c_first][(n0 + i) % 4u];
  double z[6];
  if (p->noise_kind == ORC_NOISE_UNIFORM) {
    /* (2 h + 1) 2^-16 - 1 : symmetric on (-1,1), exactly representable; component 2j from the high half */
    for (uint32_t j = 0; j < nx / 2u; ++j) {
      z[2 * j] = (double)(2u * (r[j] >> 16) + 1u) * (1.0 / 65536.0) - 1.0;
      z[2 * j + 1] = (double)(2u * (r[j] & 0xFFFFu) + 1u) * (1.0 / 65536.0) - 1.0;
    }
  } else {
    for (uint32_t j = 0; j < nx / 2u; ++j) orc_box_muller16(r[j], z + 2 * j);
  }
  if (p->noise_kind == ORC_NOISE_JUMP) {
    const double uj = (double)(r[nx / 2u] >> 16) * (1.0 / 65536.0);   /* trigger: high half of the word after the pairs */
    double nrm = 0.0;
    for (uint32_t i = 0; i < nx; ++i) nrm += z[i] * z[i];
    nrm = std::sqrt(nrm);
    const bool jump = (uj < p->noise_p[0]) && nrm > 0.0;
    for (uint32_t i = 0; i < nx; ++i) z[i] = jump ? z[i] / nrm : 0.0;
  }
  for (uint32_t i = 0; i < nx; ++i) w[i] = p->sigma_w[i] * z[i];
}

/* x_{t+1} = F(x_t, u_t)  (1) P:29.  Forward Euler, derivatives at the pre-step
 * state (D:G15); controls clamped inside F only (D:G16). */
void orc_dynamics(const orc_problem* p, const double* x, const double u[2], double* xn) {
  const double dt = p->dt;
  const double u0 = clampd(u[0], p->u_min[0], p->u_max[0]);
  const double u1 = clampd(u[1], p->u_min[1], p->u_max[1]);
  if (p->dyn == ORC_DYN_BICYCLE) {
    /* kinematic bicycle (X,Y,psi,v), u=(delta,a), wheelbase L */
    const double L = p->dyn_p[0];
    const double X = x[0], Y = x[1], psi = x[2], v = x[3];
    xn[0] = X + dt * v * std::cos(psi);
    xn[1] = Y + dt * v * std::sin(psi);
    xn[2] = psi + dt * v * std::tan(u0) / L;
    xn[3] = v + dt * u1;
  } else {
    /* single-track with linear tyres (X,Y,psi,vx,vy,r), u=(delta,Fx) */
    const double m = p->dyn_p[0], Iz = p->dyn_p[1], lf = p->dyn_p[2], lr = p->dyn_p[3];
    const double Cf = p->dyn_p[4], Cr = p->dyn_p[5], vx_floor = p->dyn_p[6];
    const double X = x[0], Y = x[1], psi = x[2], vx = x[3], vy = x[4], r = x[5];
    const double delta = u0, Fx = u1;
    const double alpha_f = delta - std::atan2(vy + lf * r, vx);
    const double alpha_r = -std::atan2(vy - lr * r, vx);
    const double Fyf = Cf * alpha_f;
    const double Fyr = Cr * alpha_r;
    const double vx_dot = (Fx - Fyf * std::sin(delta)) / m + vy * r;
    const double vy_dot = (Fyf * std::cos(delta) + Fyr) / m - vx * r;
    const double r_dot = (lf * Fyf * std::cos(delta) - lr * Fyr) / Iz;
    const double X_dot = vx * std::cos(psi) - vy * std::sin(psi);
    const double Y_dot = vx * std::sin(psi) + vy * std::cos(psi);
    xn[0] = X + dt * X_dot;
    xn[1] = Y + dt * Y_dot;
    xn[2] = psi + dt * r;
    xn[3] = std::max(vx + dt * vx_dot, vx_floor);
    xn[4] = vy + dt * vy_dot;
    xn[5] = r + dt * r_dot;
  }
}

/* First-order signed distance to the ellipse (X/a)^2+(Y/b)^2=1, + outside (D:G25). */
double orc_ellipse_offset(double a, double b, double X, double Y) {
  const double f = (X / a) * (X / a) + (Y / b) * (Y / b) - 1.0;
  const double g = std::sqrt(X * X / (a * a * a * a) + Y * Y / (b * b * b * b));
  return f / (2.0 * std::max(g, 1e-12));
}

/* Rounded-rectangle track (synthetic stand-in for the paper's track: 0.6 m wide, 10.9 m
 * centreline, corner radius 0.3 m; its layout figure P:257 is missing).  The centreline is the set
 * of points at distance rc from the box B = [-ax,ax] x [-ay,ay].  e = signed distance to the
 * centreline, + outward ("lateral deviation e(x)"). */
double orc_racing_offset(const orc_problem* p, double X, double Y) {
  const double ax = p->nom_p[0], ay = p->nom_p[1], rc = p->nom_p[2];
  const double qx = std::fabs(X) - ax, qy = std::fabs(Y) - ay;
  const double ox = std::max(qx, 0.0), oy = std::max(qy, 0.0);
  const double sd = std::sqrt(ox * ox + oy * oy) + std::min(std::max(qx, qy), 0.0);  /* signed distance to B */
  return sd - rc;
}

/* Arc length s(x) of the projection onto the centreline (Fig. 2), measured counter-clockwise
 * from (ax+rc, 0); one quadrant is folded onto the first by symmetry. */
double orc_racing_arclength(const orc_problem* p, double X, double Y) {
  const double ax = p->nom_p[0], ay = p->nom_p[1], rc = p->nom_p[2];
  const double Xa = std::fabs(X), Ya = std::fabs(Y);
  const double dx = std::max(Xa - ax, 0.0), dy = std::max(Ya - ay, 0.0);
  const double Pq = ay + rc * (kPi / 2.0) + ax;  /* quarter perimeter */
  double sq;
  if (dx > 0.0 && dy > 0.0) sq = ay + rc * std::atan2(dy, dx);             /* corner arc       */
  else if (dx > 0.0) sq = Ya;                                               /* right straight   */
  else if (dy > 0.0) sq = ay + rc * (kPi / 2.0) + (ax - Xa);                /* top straight     */
  else sq = ((ax - Xa) < (ay - Ya)) ? Ya : ay + rc * (kPi / 2.0) + (ax - Xa); /* inside B: nearest side */
  if (X >= 0.0 && Y >= 0.0) return sq;
  if (X < 0.0 && Y >= 0.0) return 2.0 * Pq - sq;
  if (X < 0.0 && Y < 0.0) return 2.0 * Pq + sq;
  return 4.0 * Pq - sq;
}

double orc_indicator_margin(const orc_problem* p, double X, double Y) {
  double m = std::numeric_limits<double>::infinity();
  for (int i = 0; i < p->n_circles; ++i) {
    const double dx = X - p->circles[3 * i + 0], dy = Y - p->circles[3 * i + 1];
    m = std::min(m, std::fabs(std::sqrt(dx * dx + dy * dy) - p->circles[3 * i + 2]));
  }
  return m;
}

/* smallest |d_i - (r_i + margin)| over the obstacles at (X,Y): distance of the hinge risk cost (circle risk of
 * orc_l) from the rim where it switches between exactly 0 and > 0.  A diagnostic for the parity tests ("exact
 * zeros must match" wherever the state is not within rounding of a rim), not part of the method. */
double orc_hinge_margin(const orc_problem* p, double X, double Y) {
  double m = std::numeric_limits<double>::infinity();
  for (int i = 0; i < p->n_circles; ++i) {
    const double dx = X - p->circles[3 * i + 0], dy = Y - p->circles[3 * i + 1];
    m = std::min(m, std::fabs(std::sqrt(dx * dx + dy * dy) - (p->circles[3 * i + 2] + p->risk_p[1])));
  }
  return m;
}

namespace {
/* state part of the nominal running cost; q "can take an arbitrary form" P:45 */
double q_state(const orc_problem* p, const double* x) {
  if (p->nominal == ORC_NOM_RACING) {
    /* (20) P:164: q = c1 mu_bdry + c2 mu_obs + c3 q_dev, q_dev = e^2 */
    const double hw = p->nom_p[3], c1 = p->nom_p[4], c2 = p->nom_p[5], c3 = p->nom_p[6];
    const double e = orc_racing_offset(p, x[0], x[1]);
    const double d = hw - std::fabs(e);      /* signed distance from the nearest boundary, + on track */
    const double mu_bdry = std::max(0.0, std::atan(-100.0 * d) / kPi + 0.5);                 /* (21) P:227 */
    double mu_obs = 0.0;                                                                      /* (22) P:232 */
    for (int i = 0; i < p->n_circles; ++i) {
      const double dx = x[0] - p->circles[3 * i + 0], dy = x[1] - p->circles[3 * i + 1];
      if (std::sqrt(dx * dx + dy * dy) < p->circles[3 * i + 2]) mu_obs += 1.0;
    }
    return c1 * mu_bdry + c2 * mu_obs + c3 * e * e;
  }
  if (p->nominal == ORC_NOM_GOAL) {
    const double w = p->nom_p[0], gx = p->nom_p[1], gy = p->nom_p[2];
    return w * ((x[0] - gx) * (x[0] - gx) + (x[1] - gy) * (x[1] - gy));
  }
  const double a = p->nom_p[0], b = p->nom_p[1], half_w = p->nom_p[2];
  const double w_lat = p->nom_p[3], w_v = p->nom_p[4], v_ref = p->nom_p[5], w_bdry = p->nom_p[6];
  const double e = orc_ellipse_offset(a, b, x[0], x[1]);
  const double v = x[3]; /* bicycle v, single-track vx */
  const double over = std::max(0.0, std::fabs(e) - half_w);
  return w_lat * e * e + w_v * (v - v_ref) * (v - v_ref) + w_bdry * over * over;
}
}  // namespace

double orc_q(const orc_problem* p, const double* x) { return q_state(p, x); }

/* phi(x) = w_phi * q_state(x)  (D:G18); racing: (23) P:239 phi = c4 - c5 s(x), s = distance travelled
 * along the centreline by the end of the horizon, i.e. s(x_T) - s(x_0) wrapped to (-P/2, P/2]. */
double orc_phi(const orc_problem* p, const double* x, const double* x0) {
  if (p->nominal == ORC_NOM_RACING) {
    const double P = 4.0 * (p->nom_p[1] + p->nom_p[2] * (kPi / 2.0) + p->nom_p[0]);
    double ds = orc_racing_arclength(p, x[0], x[1]) - orc_racing_arclength(p, x0[0], x0[1]);
    if (ds > 0.5 * P) ds -= P;
    if (ds < -0.5 * P) ds += P;
    return p->nom_p[7] - p->nom_p[8] * ds;
  }
  const double w_phi = p->nominal == ORC_NOM_GOAL ? p->nom_p[3] : p->nom_p[7];
  return w_phi * q_state(p, x);
}

/* bilinear lookup between cell centres, clamp-to-edge (D:G26) */
double orc_bilinear(const orc_problem* p, double X, double Y) {
  const double gx = (X - p->map_ox) / p->map_res - 0.5;
  const double gy = (Y - p->map_oy) / p->map_res - 0.5;
  const double fx0 = std::floor(gx), fy0 = std::floor(gy);
  const double fx = gx - fx0, fy = gy - fy0;
  auto cl = [](double i, int n) { return (int)std::min(std::max(i, 0.0), (double)(n - 1)); };
  const int ix0 = cl(fx0, p->map_w), ix1 = cl(fx0 + 1.0, p->map_w);
  const int iy0 = cl(fy0, p->map_h), iy1 = cl(fy0 + 1.0, p->map_h);
  const double c00 = p->costmap[(size_t)iy0 * p->map_w + ix0];
  const double c01 = p->costmap[(size_t)iy0 * p->map_w + ix1];
  const double c10 = p->costmap[(size_t)iy1 * p->map_w + ix0];
  const double c11 = p->costmap[(size_t)iy1 * p->map_w + ix1];
  return (1.0 - fy) * ((1.0 - fx) * c00 + fx * c01) + fy * ((1.0 - fx) * c10 + fx * c11);
}

/* l(x~) of (9) P:93, "running cost of arbitrary form" P:95. */
double orc_l(const orc_problem* p, const double* x) {
  if (p->risk == ORC_RISK_CIRCLES) {
    /* sum_i weight * max(0, r_i + margin - d_i)^2, d_i = |(X,Y)-c_i|  (D:G22) */
    const double weight = p->risk_p[0], margin = p->risk_p[1];
    double l = 0.0;
    for (int i = 0; i < p->n_circles; ++i) {
      const double dx = x[0] - p->circles[3 * i + 0];
      const double dy = x[1] - p->circles[3 * i + 1];
      const double d = std::sqrt(dx * dx + dy * dy);
      const double pen = std::max(0.0, p->circles[3 * i + 2] + margin - d);
      l += weight * pen * pen;
    }
    return l;
  }
  if (p->risk == ORC_RISK_COSTMAP) return p->risk_p[0] * orc_bilinear(p, x[0], x[1]);
  if (p->risk == ORC_RISK_NOMINAL) return q_state(p, x);   /* "l(x~) = q(x~)" P:247 */
  /* test-only: weight * x[index] */
  return p->risk_p[0] * x[(int)p->risk_p[1]];
}

/* k_tail = ceil((1-alpha) M), robust to fp64 representation of alpha (D:G11). */
int32_t orc_tail_count(double alpha, int32_t M) {
  int32_t k = (int32_t)std::ceil((1.0 - alpha) * (double)M - 1e-9);
  return std::min(std::max(k, 1), M);
}

/* Alg.1 l.25-26 P:204-207: P = upper (1-alpha) quantile set, CVaR = Average(P).
 * Written as the definition: full sort, mean of the k_tail largest. */
double orc_cvar_topk(const double* L, int32_t M, int32_t k_tail) {
  std::vector<double> s(L, L + M);
  std::sort(s.begin(), s.end(), std::greater<double>());
  double sum = 0.0;
  for (int32_t i = 0; i < k_tail; ++i) sum += s[i];
  return sum / (double)k_tail;
}

/* Literal (11)-(13) P:101-111: VaR = min{t : P(L<=t) >= alpha} on the empirical
 * distribution, CVaR = mean of all samples >= VaR (N_o of them).  Cross-check of
 * the reading D:G11; agrees with top-k when there is no tie at VaR and
 * (1-alpha)M is not an integer. */
double orc_cvar_literal12(const double* L, int32_t M, double alpha) {
  std::vector<double> s(L, L + M);
  std::sort(s.begin(), s.end());
  double var = s[M - 1];
  for (int32_t i = 0; i < M; ++i) {
    /* number of samples <= s[i] */
    int32_t cnt = (int32_t)(std::upper_bound(s.begin(), s.end(), s[i]) - s.begin());
    if ((double)cnt >= alpha * (double)M - 1e-9) { var = s[i]; break; }
  }
  double sum = 0.0; int32_t n_o = 0;
  for (int32_t i = 0; i < M; ++i) if (L[i] >= var) { sum += L[i]; ++n_o; }
  return sum / (double)n_o;
}

/* (18)-(19) P:144-148 with the mean read as (1/M) sum (D:G7). */
void orc_sensitivity_scale(const double* L, int32_t M, double B, double* La) {
  double Lbar = 0.0;
  for (int32_t m = 0; m < M; ++m) Lbar += L[m];
  Lbar /= (double)M;
  for (int32_t m = 0; m < M; ++m) La[m] = B * (L[m] - Lbar) + Lbar;
}

namespace {

/* O1 for one control sample k (Alg.1 l.3-29 P:175-213). */
void one_sample(const orc_problem* p, const double* x0_in, const double* v, uint64_t iteration,
                int32_t k, int32_t k_tail, int32_t K0,
                double* u_out, double* S_out, double* cvar_out, double* Stil_out,
                double* L_out, double* xT_out, double* xnom_out, double* margin_out) {
  const int nx = orc_nx(p->dyn);
  const int T = p->T, M = p->M;
  const uint32_t key[2] = {(uint32_t)(p->seed & 0xFFFFFFFFull), (uint32_t)(p->seed >> 32)};

  /* x0: single-track vx floored on entry (D: models) */
  double x0[6];
  for (int i = 0; i < nx; ++i) x0[i] = x0_in[i];
  if (p->dyn == ORC_DYN_SINGLE_TRACK) x0[3] = std::max(x0[3], p->dyn_p[6]);

  /* O1a: eps^k ~ N(0,Sigma_eps) (2c) P:42, Alg.1 l.4 P:179;
   * u = v + eps for k < (1-eta)K (l.8), u = eps otherwise (l.10) P:183-187 */
  std::vector<double> u((size_t)T * 2);
  for (int t = 0; t < T; ++t) {
    uint32_t ctr[4], r[4];
    orc_counter((uint32_t)k, 0u, (uint32_t)t, 1u, 0u, ORC_STREAM_EPS, iteration, ctr);
    orc_philox4x32_10(ctr, key, r);
    double z[2];
    orc_box_muller(r[0], r[1], z);
    for (int i = 0; i < 2; ++i) {
      const double eps = p->sigma_eps[i] * z[i];
      u[2 * t + i] = (k < K0 ? v[2 * t + i] : 0.0) + eps;
    }
  }

  /* O1b: nominal rollout and cost (3) P:47 / (16) P:129, Alg.1 l.11-15 P:188-193 */
  double x[6], xn[6];
  for (int i = 0; i < nx; ++i) x[i] = x0[i];
  double S = 0.0;
  const bool want_margin = margin_out && p->nominal == ORC_NOM_RACING;
  double mg = std::numeric_limits<double>::infinity();
  for (int t = 0; t < T; ++t) {
    if (want_margin) mg = std::min(mg, orc_indicator_margin(p, x[0], x[1]));
    double ctrl = 0.0;
    for (int i = 0; i < 2; ++i)
      if (p->sigma_eps[i] > 0.0)
        ctrl += v[2 * t + i] * u[2 * t + i] / (p->sigma_eps[i] * p->sigma_eps[i]);
    S += orc_q(p, x) + p->gamma * ctrl;
    orc_dynamics(p, x, &u[2 * t], xn);
    for (int i = 0; i < nx; ++i) x[i] = xn[i];
  }
  S += orc_phi(p, x, x0);
  if (margin_out) margin_out[0] = mg;

  /* O1c: M noisy rollouts (6) P:63 from x~_0 = x_0 P:109, risk cost (9) P:93,
   * Alg.1 l.16-21 P:194-199; driven by the sampled u^k (D:G6) */
  std::vector<double> Lk((size_t)M), La((size_t)M);
  for (int m = 0; m < M; ++m) {
    double xt[6];
    for (int i = 0; i < nx; ++i) xt[i] = x0[i];
    double L = 0.0;
    double mgm = std::numeric_limits<double>::infinity();
    for (int t = 0; t < T; ++t) {
      if (margin_out && p->risk == ORC_RISK_NOMINAL && p->nominal == ORC_NOM_RACING)
        mgm = std::min(mgm, orc_indicator_margin(p, xt[0], xt[1]));
      if (margin_out && p->risk == ORC_RISK_CIRCLES)
        mgm = std::min(mgm, orc_hinge_margin(p, xt[0], xt[1]));
      L += orc_l(p, xt);
      double w[6];
      orc_state_noise(p, (uint32_t)k, (uint32_t)m, (uint32_t)t, ORC_STREAM_W, iteration, w);
      orc_dynamics(p, xt, &u[2 * t], xn);
      for (int i = 0; i < nx; ++i) xt[i] = xn[i] + w[i];
      if (p->dyn == ORC_DYN_SINGLE_TRACK) xt[3] = std::max(xt[3], p->dyn_p[6]);
    }
    Lk[m] = L;
    if (margin_out) margin_out[1 + m] = mgm;
    if (L_out) L_out[m] = L;
    if (xT_out) for (int i = 0; i < nx; ++i) xT_out[(size_t)m * nx + i] = xt[i];
  }

  /* O1d: sensitivity scaling (18)-(19), Alg.1 l.24 P:204 */
  orc_sensitivity_scale(Lk.data(), M, p->B, La.data());
  /* O1e: CVaR, Alg.1 l.25-26 */
  const double cvar = orc_cvar_topk(La.data(), M, k_tail);
  /* O1f: soft filter (14)-(16) P:120-130, Alg.1 l.27-29 (strict >, else S~ = S; D:G10) */
  const double Stil = S + (cvar > p->C_u ? p->A * cvar : 0.0);

  if (u_out) for (int i = 0; i < 2 * T; ++i) u_out[i] = u[i];
  if (S_out) *S_out = S;
  if (cvar_out) *cvar_out = cvar;
  if (Stil_out) *Stil_out = Stil;
  if (xnom_out) for (int i = 0; i < nx; ++i) xnom_out[i] = x[i];
}

}  // namespace

int orc_rollout_costs(const orc_problem* p, const double* x0, const double* v,
                      uint64_t iteration, int32_t k_begin, int32_t k_end, int32_t n_threads,
                      double* u, double* S, double* cvar, double* S_tilde, double* L, double* xT,
                      double* x_nom, double* margin) {
  if (!p || !x0 || !v || k_begin < 0 || k_end > p->K || k_begin > k_end) return 1;
  const int nx = orc_nx(p->dyn);
  const int32_t k_tail = orc_tail_count(p->alpha, p->M);                       /* O0 */
  const int32_t K0 = (int32_t)std::ceil((1.0 - p->eta) * (double)p->K - 1e-9);
  const size_t T = (size_t)p->T, M = (size_t)p->M;
  auto work = [&](int32_t kb, int32_t ke) {
    for (int32_t k = kb; k < ke; ++k) {
      const size_t i = (size_t)(k - k_begin);
      one_sample(p, x0, v, iteration, k, k_tail, K0,
                 u ? u + i * T * 2 : nullptr, S ? S + i : nullptr, cvar ? cvar + i : nullptr,
                 S_tilde ? S_tilde + i : nullptr, L ? L + i * M : nullptr,
                 xT ? xT + i * M * nx : nullptr, x_nom ? x_nom + i * nx : nullptr,
                 margin ? margin + i * (M + 1) : nullptr);
    }
  };
  const int32_t n = k_end - k_begin;
  if (n_threads <= 1 || n < 2) { work(k_begin, k_end); return 0; }
  std::vector<std::thread> th;
  const int32_t nt = std::min(n_threads, n);
  for (int32_t i = 0; i < nt; ++i) {
    const int32_t kb = k_begin + (int32_t)((int64_t)n * i / nt);
    const int32_t ke = k_begin + (int32_t)((int64_t)n * (i + 1) / nt);
    th.emplace_back(work, kb, ke);
  }
  for (auto& t : th) t.join();
  return 0;
}

/* O2: (17) P:134 / (5) P:55 with beta~ = min S~ ; O3: (4) P:51, then clamp (D:G16). */
int orc_weights_update(const orc_problem* p, const double* S_tilde, const double* u,
                       double* v_plus, double* w_out, double* Z_out, double* beta_out) {
  const int K = p->K, T = p->T;
  double beta = std::numeric_limits<double>::infinity();
  for (int k = 0; k < K; ++k) beta = std::min(beta, S_tilde[k]);
  std::vector<double> w((size_t)K);
  double Z = 0.0;
  for (int k = 0; k < K; ++k) {
    w[k] = std::exp(-(S_tilde[k] - beta) / p->lambda);
    Z += w[k];
  }
  for (int t = 0; t < T; ++t)
    for (int i = 0; i < 2; ++i) {
      double num = 0.0;
      for (int k = 0; k < K; ++k) num += w[k] * u[((size_t)k * T + t) * 2 + i];
      if (v_plus) v_plus[2 * t + i] = clampd(num / Z, p->u_min[i], p->u_max[i]);
    }
  if (w_out) for (int k = 0; k < K; ++k) w_out[k] = w[k];
  if (Z_out) *Z_out = Z;
  if (beta_out) *beta_out = beta;
  return 0;
}

int orc_step(const orc_problem* p, const double* x0, const double* v, uint64_t iteration,
             int32_t n_threads, double* v_plus) {
  std::vector<double> u((size_t)p->K * p->T * 2), Stil((size_t)p->K);
  int rc = orc_rollout_costs(p, x0, v, iteration, 0, p->K, n_threads, u.data(), nullptr, nullptr,
                             Stil.data(), nullptr, nullptr, nullptr, nullptr);
  if (rc) return rc;
  return orc_weights_update(p, Stil.data(), u.data(), v_plus, nullptr, nullptr, nullptr);
}

/* Alg.1 l.32 P:218 ExecuteCommand(v+_0) on a simulated plant: the disturbed
 * dynamics (6) with the PLANT stream (BASELINE config 4). */
void orc_plant_step(const orc_problem* p, const double* x0, const double u0[2],
                    uint64_t iteration, double* x_next) {
  const int nx = orc_nx(p->dyn);
  double x[6], xn[6], w[6];
  for (int i = 0; i < nx; ++i) x[i] = x0[i];
  if (p->dyn == ORC_DYN_SINGLE_TRACK) x[3] = std::max(x[3], p->dyn_p[6]);
  orc_dynamics(p, x, u0, xn);
  orc_state_noise(p, 0u, 0u, 0u, ORC_STREAM_PLANT, iteration, w);
  for (int i = 0; i < nx; ++i) x_next[i] = xn[i] + w[i];
  if (p->dyn == ORC_DYN_SINGLE_TRACK) x_next[3] = std::max(x_next[3], p->dyn_p[6]);
}

/* Alg.1 l.33 P:220 v = v+, plus the warm-start shift config 4 asks for (D:G19). */
void orc_shift(const double* v_plus, int32_t T, double* v_next) {
  for (int t = 0; t < T - 1; ++t) {
    v_next[2 * t] = v_plus[2 * (t + 1)];
    v_next[2 * t + 1] = v_plus[2 * (t + 1) + 1];
  }
  v_next[2 * (T - 1)] = v_plus[2 * (T - 1)];
  v_next[2 * (T - 1) + 1] = v_plus[2 * (T - 1) + 1];
}

}  // extern "C"
