// Sanitizer driver for the oracle (-fsanitize=address,undefined on the oracle).
// Compiled together with oracle/ra_mppi_oracle.cpp by tests/test_oracle_sanitizers.py; runs every exported
// function on small problems that cover both models, all cost kinds and all noise kinds with ragged sizes.
// Exit code 0 and no sanitizer report = pass.  Values are not checked here (the pins do that).
#include <cmath>
#include <cstdio>
#include <vector>

#include "ra_mppi_oracle.h"

static orc_problem base(int K, int M, int T) {
  orc_problem p{};
  p.K = K; p.M = M; p.T = T; p.dt = 0.05;
  p.dyn = ORC_DYN_BICYCLE; p.dyn_p[0] = 0.33;
  p.u_min[0] = -0.35; p.u_max[0] = 0.35; p.u_min[1] = -3.0; p.u_max[1] = 3.0;
  p.sigma_eps[0] = 0.1; p.sigma_eps[1] = 0.5;
  const double sw[6] = {0.02, 0.02, 0.01, 0.05, 0.05, 0.05};
  for (int i = 0; i < 6; ++i) p.sigma_w[i] = sw[i];
  p.alpha = 0.9; p.lambda = 1.0; p.gamma = 1.0; p.A = 1.0; p.B = 1.5; p.C_u = 0.0; p.eta = 0.3;
  p.nominal = ORC_NOM_GOAL; p.nom_p[0] = 1.0; p.nom_p[1] = 18.0; p.nom_p[2] = 18.0; p.nom_p[3] = 1.0;
  p.risk = ORC_RISK_CIRCLES; p.risk_p[0] = 1000.0; p.risk_p[1] = 0.2;
  p.seed = 0x0123456789ABCDEFull;
  return p;
}

static int run(const orc_problem& p, const std::vector<double>& x0, bool margin) {
  const int nx = orc_nx(p.dyn);
  std::vector<double> v((size_t)p.T * 2);
  for (size_t i = 0; i < v.size(); ++i) v[i] = 0.05 * std::sin(0.7 * (double)i);
  const size_t K = (size_t)p.K, M = (size_t)p.M, T = (size_t)p.T;
  std::vector<double> u(K * T * 2), S(K), cv(K), St(K), L(K * M), xT(K * M * nx), xn(K * nx), mg(K * (M + 1));
  int rc = orc_rollout_costs(&p, x0.data(), v.data(), 3, 0, p.K, 3, u.data(), S.data(), cv.data(), St.data(), L.data(),
                             xT.data(), xn.data(), margin ? mg.data() : nullptr);
  /* a sub-range with every optional output absent */
  if (p.K >= 3) rc |= orc_rollout_costs(&p, x0.data(), v.data(), 3, 1, p.K - 1, 1, nullptr, nullptr, nullptr, St.data() + 1,
                                        nullptr, nullptr, nullptr, nullptr);
  std::vector<double> vp(T * 2), w(K), vnext(T * 2), xp(6);
  double Z = 0, beta = 0;
  rc |= orc_weights_update(&p, St.data(), u.data(), vp.data(), w.data(), &Z, &beta);
  rc |= orc_step(&p, x0.data(), v.data(), 4, 2, vp.data());
  orc_plant_step(&p, x0.data(), vp.data(), 4, xp.data());
  orc_shift(vp.data(), p.T, vnext.data());
  const int kt = orc_tail_count(p.alpha, p.M);
  std::vector<double> La(M);
  orc_sensitivity_scale(L.data(), p.M, p.B, La.data());
  const double a = orc_cvar_topk(La.data(), p.M, kt), b = orc_cvar_literal12(La.data(), p.M, p.alpha);
  if (!(std::isfinite(a) && std::isfinite(b) && std::isfinite(Z) && Z >= 1.0)) rc |= 2;
  for (double x : vp) if (!std::isfinite(x)) rc |= 4;
  return rc;
}

int main() {
  int rc = 0;
  std::vector<double> circles = {2.0, 2.2, 0.4, 5.0, 5.0, 0.5, 9.0, 5.0, 0.3};
  {  /* bicycle, goal cost, circle risk, Gaussian noise, M = 1 and a ragged M */
    orc_problem p = base(7, 1, 5);
    p.circles = circles.data(); p.n_circles = 3;
    rc |= run(p, {1.0, 1.0, 0.785, 2.0}, true);
    p.M = 37; p.K = 5; p.alpha = 0.5;
    rc |= run(p, {1.0, 1.0, 0.785, 2.0}, true);
    p.n_circles = 0; p.circles = nullptr;           /* empty obstacle set */
    rc |= run(p, {1.0, 1.0, 0.785, 2.0}, true);
  }
  {  /* single-track, ellipse track, jump noise (n_x + 2 words per step), odd horizon */
    orc_problem p = base(6, 9, 7);
    p.dyn = ORC_DYN_SINGLE_TRACK;
    const double dp[7] = {4.0, 0.05, 0.17, 0.17, 30.0, 30.0, 0.5};
    for (int i = 0; i < 7; ++i) p.dyn_p[i] = dp[i];
    p.u_min[1] = -10.0; p.u_max[1] = 10.0; p.sigma_eps[1] = 2.0; p.dt = 0.02;
    p.nominal = ORC_NOM_ELLIPSE_TRACK;
    const double np_[8] = {10.0, 6.0, 1.0, 5.0, 2.0, 4.0, 1000.0, 1.0};
    for (int i = 0; i < 8; ++i) p.nom_p[i] = np_[i];
    std::vector<double> c2 = {10.0, 0.4, 0.3, 9.8, 1.0, 0.2};
    p.circles = c2.data(); p.n_circles = 2;
    p.noise_kind = ORC_NOISE_JUMP; p.noise_p[0] = 0.3;
    rc |= run(p, {10.0, 0.0, 1.5707963, 0.3, 0.0, 0.0}, true);
    p.noise_kind = ORC_NOISE_GAUSSIAN;
    rc |= run(p, {10.0, 0.0, 1.5707963, 3.0, 0.0, 0.0}, false);
  }
  {  /* costmap risk, uniform noise; positions that leave the map exercise clamp-to-edge */
    orc_problem p = base(5, 8, 30);
    std::vector<double> map(6 * 9);
    for (size_t i = 0; i < map.size(); ++i) map[i] = (double)(i % 5) / 4.0;
    p.risk = ORC_RISK_COSTMAP; p.costmap = map.data(); p.map_h = 6; p.map_w = 9; p.map_res = 0.5;
    p.map_ox = 0.5; p.map_oy = 0.25; p.noise_kind = ORC_NOISE_UNIFORM;
    rc |= run(p, {1.0, 1.0, 0.785, 4.0}, false);
    rc |= run(p, {-3.0, 9.0, 2.5, 4.0}, false);
  }
  {  /* the paper's racing costs (20)-(23) with l = q, linear test risk */
    orc_problem p = base(4, 11, 6);
    p.nominal = ORC_NOM_RACING;
    const double np_[9] = {1.5, 0.7537, 0.3, 0.3, 2.0, 1.0, 0.1, 0.6, 2.0};
    for (int i = 0; i < 9; ++i) p.nom_p[i] = np_[i];
    std::vector<double> c3 = {0.2, -1.05, 0.1, 1.8, 0.1, 0.1};
    p.circles = c3.data(); p.n_circles = 2; p.risk = ORC_RISK_NOMINAL; p.dt = 0.02; p.dyn_p[0] = 0.093;
    rc |= run(p, {0.0, -1.0537, 0.0, 1.5}, true);
    p.risk = ORC_RISK_LINEAR_STATE; p.risk_p[0] = -1.0; p.risk_p[1] = 3.0;
    rc |= run(p, {0.0, -1.0537, 0.0, 1.5}, false);
  }
  uint32_t ctr[4], out[4]; const uint32_t key[2] = {1u, 2u};
  orc_counter(0xFFFFFFFFu, 0xFFFFFFFFu, 0x7FFFFFFFu, 2u, 1u, 2u, ~0ull, ctr);
  orc_philox4x32_10(ctr, key, out);
  double z[2];
  orc_box_muller(out[0], out[1], z);
  orc_box_muller(0xFFFFFFFFu, 0u, z);
  std::printf("oracle sanitizer run: rc=%d\n", rc);
  return rc;
}
