// Vehicle models and cost functions of the BASELINE configs (device side, fp32).
// Dynamics: x_{t+1} = F(x_t, u_t) (1) PAPER.md:29, forward Euler with derivatives at the
// pre-step state; controls clamped inside F.  Positions are integrated in a frame centred at
// x0's position (exactly translation-invariant models), which keeps fp32 rounding of the
// Euler sums at the scale of the travelled distance instead of the world coordinate.
#pragma once
#include "ra_params.cuh"

namespace ra {

__device__ __forceinline__ float clampf(float x, float lo, float hi) { return fminf(fmaxf(x, lo), hi); }

// sin/cos by three-term Cody-Waite reduction to [-pi/4, pi/4] and FMA-pipe polynomials.
// Valid (<= 2 ulp) for |x| < ~6000 rad; yaw angles here stay within a few turns.
__device__ __forceinline__ void sincos_cw(float x, float& s, float& c) {
  // round-to-nearest by the 1.5*2^23 trick (FMA pipe; no FRND/F2I on the XU pipe): the low mantissa
  // bits of jm hold the integer, valid for |x| < 2^21 quarter-turns
  const float jm = fmaf(x, 0.636619747f, 12582912.0f);
  const float j = jm - 12582912.0f;
  float r = fmaf(j, -1.5703125f, x);
  r = fmaf(j, -4.837512969970703e-4f, r);
  r = fmaf(j, -7.549790126404332e-8f, r);
  const float r2 = r * r;
  float ps = 2.75573192e-6f;            //  1/9!
  ps = fmaf(ps, r2, -1.98412698e-4f);   // -1/7!
  ps = fmaf(ps, r2, 8.33333333e-3f);    //  1/5!
  ps = fmaf(ps, r2, -1.66666667e-1f);   // -1/3!
  const float sr = fmaf(r * r2, ps, r);
  float pc = 2.48015873e-5f;            //  1/8!
  pc = fmaf(pc, r2, -1.38888889e-3f);   // -1/6!
  pc = fmaf(pc, r2, 4.16666667e-2f);    //  1/4!
  pc = fmaf(pc, r2, -0.5f);
  const float cr = fmaf(pc, r2, 1.0f);
  const int q = __float_as_int(jm);
  const float cs = (q & 1) ? -sr : cr;
  const float sn = (q & 1) ? cr : sr;
  c = (q & 2) ? -cs : cs;
  s = (q & 2) ? -sn : sn;
}

// sin/cos of the yaw angle inside the K*M*T noisy rollouts: MUFU.SIN / MUFU.COS on the angle itself (SASS: one
// FMUL.RZ by 1/(2 pi) feeding both, the unit works in turns and drops whole turns exactly).  The rollout kernel
// starts every realisation from a yaw reduced to [-pi, pi) (reduce_yaw below), so within the horizon |psi| stays at a
// few turns at most: the multiply is then good to 2^-24 |psi| (<= 4e-7 rad per turn of winding) on top of the unit's
// 2^-21.4 abs error -- per Euler step <= dt v 1e-6 ~ 2e-7 m of position, at the half-ulp (2.4e-7 m for |X| in [4,8) m)
// that the fp32 position sum rounds by anyway; 3 instructions instead of 25 (round 1 reduced every step: 7).
// The K*T nominal rollout and the plant keep sincos_cw.
__device__ __forceinline__ void sincos_mufu(float x, float& s, float& c) {
  s = __sinf(x);
  c = __cosf(x);
}

// psi = psi_rel + n 2 pi with psi_rel in [-pi, pi]: once per thread at rollout start; restore_yaw undoes it for output.
__device__ __forceinline__ float reduce_yaw(float psi, float& n_turns) {
  n_turns = rintf(psi * 0.159154943f);
  return fmaf(n_turns, -1.9353071795864769e-3f, fmaf(n_turns, -6.28125f, psi));
}
__device__ __forceinline__ float restore_yaw(float psi_rel, float n_turns) {
  return fmaf(n_turns, 6.28125f, fmaf(n_turns, 1.9353071795864769e-3f, psi_rel));
}

// atan2(y, x) for x > 0 (the single-track model floors vx at a positive value): one MUFU.RCP and
// a degree-8 odd polynomial in z = min(|y|,x)/max(|y|,x) (max error 1.3e-7 rad in fp32, fitted on
// Chebyshev nodes; the linear coefficient is exactly 1 so small slip angles keep relative accuracy).
__device__ __forceinline__ float atan2_posx(float y, float x) {
  const float ay = fabsf(y);
  const float den = fmaxf(ay, x);
  float inv;
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(inv) : "f"(den));
  const float z = fminf(ay, x) * inv;
  const float s = z * z;
  float p = 0.0028340641874819994f;
  p = fmaf(p, s, -0.016005029901862144f);
  p = fmaf(p, s, 0.042587608098983765f);
  p = fmaf(p, s, -0.07495445758104324f);
  p = fmaf(p, s, 0.10636754333972931f);
  p = fmaf(p, s, -0.14202570915222168f);
  p = fmaf(p, s, 0.19992484152317047f);
  p = fmaf(p, s, -0.3333306610584259f);
  p = fmaf(p * s, z, z);                       // z (1 + s P(s))
  const float r = (ay > x) ? 1.57079632679489662f - p : p;
  return copysignf(r, y);
}

// Control effects: everything F needs from u^k_t that is the same for all M realisations,
// computed once per (k,t) by the sampling kernel.
//   bicycle:       (dt tan(delta_c)/L, dt a_c, -, -)
//   single-track:  (delta_c, Fx_c, sin delta_c, cos delta_c)
template <int DYN>
__device__ __forceinline__ float4 control_effect(const Params& p, float u0, float u1) {
  const float d = clampf(u0, p.u_min[0], p.u_max[0]);
  const float a = clampf(u1, p.u_min[1], p.u_max[1]);
  if constexpr (DYN == DYN_BICYCLE) {
    return make_float4(p.dyn_q[0] * tanf(d), p.dt * a, 0.0f, 0.0f);   // dyn_q[0] = dt / L (host, fp64)
  } else {
    float s, c;
    sincos_cw(d, s, c);
    return make_float4(d, a, s, c);
  }
}

template <int DYN> struct StateDim { static constexpr int value = DYN == DYN_SINGLE_TRACK ? 6 : 4; };

// One Euler step in the x0-centred frame.  x: (X,Y,psi,v) or (X,Y,psi,vx,vy,r).
template <int DYN, bool FAST = false>
__device__ __forceinline__ void dynamics_step(const Params& p, float (&x)[StateDim<DYN>::value],
                                              const float4 ce) {
  float s, c;
  if constexpr (FAST) sincos_mufu(x[2], s, c);
  else sincos_cw(x[2], s, c);
  if constexpr (DYN == DYN_BICYCLE) {
    const float dv = p.dt * x[3];
    x[0] = fmaf(dv, c, x[0]);
    x[1] = fmaf(dv, s, x[1]);
    x[2] = fmaf(x[3], ce.x, x[2]);
    x[3] = x[3] + ce.y;
  } else {
    const float m_inv = p.dyn_q[0], iz_inv = p.dyn_q[1];  // 1/m, 1/Iz (host-computed)
    const float lf = p.dyn_p[2], lr = p.dyn_p[3], Cf = p.dyn_p[4], Cr = p.dyn_p[5];
    const float vx = x[3], vy = x[4], r = x[5];
    const float alpha_f = ce.x - atan2_posx(fmaf(lf, r, vy), vx);   // vx >= vx_floor > 0
    const float alpha_r = -atan2_posx(fmaf(-lr, r, vy), vx);
    const float Fyf = Cf * alpha_f, Fyr = Cr * alpha_r;
    const float vx_dot = fmaf(vy, r, (ce.y - Fyf * ce.z) * m_inv);
    const float vy_dot = fmaf(-vx, r, fmaf(Fyf, ce.w, Fyr) * m_inv);
    const float r_dot = (lf * Fyf * ce.w - lr * Fyr) * iz_inv;
    const float X_dot = vx * c - vy * s;
    const float Y_dot = fmaf(vx, s, vy * c);
    x[0] = fmaf(p.dt, X_dot, x[0]);
    x[1] = fmaf(p.dt, Y_dot, x[1]);
    x[2] = fmaf(p.dt, r, x[2]);
    x[3] = fmaxf(fmaf(p.dt, vx_dot, vx), p.dyn_p[6]);
    x[4] = fmaf(p.dt, vy_dot, vy);
    x[5] = fmaf(p.dt, r_dot, r);
  }
}

// ---- the paper's own racing costs (20)-(23), on a rounded-rectangle track -------
// nom_p = {ax, ay, rc, half_w, c1, c2, c3, c4, c5}; centreline = points at distance rc from the box
// [-ax,ax] x [-ay,ay].  e = lateral deviation (+ outward), d = half_w - |e| (+ on the track).
__device__ __forceinline__ float racing_offset(const Params& p, float X, float Y) {
  const float qx = fabsf(X) - p.nom_p[0], qy = fabsf(Y) - p.nom_p[1];
  const float ox = fmaxf(qx, 0.0f), oy = fmaxf(qy, 0.0f);
  float outside;
  asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(outside) : "f"(fmaf(ox, ox, oy * oy)));
  return outside + fminf(fmaxf(qx, qy), 0.0f) - p.nom_p[2];
}

// c1 mu_bdry + c3 e^2 : the smooth part of (20); mu_bdry = max(0, atan(-100 d)/pi + 1/2)  (21)
__device__ __forceinline__ float racing_smooth_cost(const Params& p, float X, float Y) {
  const float e = racing_offset(p, X, Y);
  const float d = p.nom_p[3] - fabsf(e);
  const float mu = fmaxf(0.0f, fmaf(atan2_posx(-100.0f * d, 1.0f), 0.318309886183790672f, 0.5f));
  return fmaf(p.nom_p[4], mu, p.nom_p[6] * e * e);
}

// s(x): arc length of the projection onto the centreline, counter-clockwise from (ax+rc, 0)
__device__ __forceinline__ float racing_arclength(const Params& p, float X, float Y) {
  const float ax = p.nom_p[0], ay = p.nom_p[1], rc = p.nom_p[2];
  const float Xa = fabsf(X), Ya = fabsf(Y);
  const float dx = fmaxf(Xa - ax, 0.0f), dy = fmaxf(Ya - ay, 0.0f);
  const float quarter_arc = rc * 1.57079632679489662f;
  const float Pq = ay + quarter_arc + ax;
  float sq;
  if (dx > 0.0f && dy > 0.0f) sq = fmaf(rc, atan2_posx(dy, dx), ay);
  else if (dx > 0.0f) sq = Ya;
  else if (dy > 0.0f) sq = ay + quarter_arc + (ax - Xa);
  else sq = ((ax - Xa) < (ay - Ya)) ? Ya : ay + quarter_arc + (ax - Xa);
  if (X >= 0.0f) return Y >= 0.0f ? sq : 4.0f * Pq - sq;
  return Y >= 0.0f ? 2.0f * Pq - sq : 2.0f * Pq + sq;
}

// Nominal running cost q(x) (state part; "arbitrary form" PAPER.md:45) at absolute position
// (X, Y) = frame origin + x[0..1]; v = x[3].  BASELINE configs 0/3 (goal) and 1/2/4 (track).
template <int NOM>
__device__ __forceinline__ float nominal_cost(const Params& p, float Xabs, float Yabs, float v) {
  if constexpr (NOM == NOM_GOAL) {
    const float dx = Xabs - p.nom_p[1], dy = Yabs - p.nom_p[2];
    return p.nom_p[0] * fmaf(dx, dx, dy * dy);
  } else if constexpr (NOM == NOM_RACING) {
    // (20): c1 mu_bdry + c2 mu_obs + c3 e^2 with the indicator obstacle cost (22) (K*T evaluations only)
    float q = racing_smooth_cost(p, Xabs, Yabs);
    for (int i = 0; i < p.n_circles; ++i) {
      const float4 c = __ldg(p.circles + i);
      const float dx = Xabs - c.x, dy = Yabs - c.y;
      if (fmaf(dx, dx, dy * dy) < c.w * c.w) q += p.nom_p[5];   // bare radius: (22) has no margin
    }
    return q;
  } else {
    // first-order signed offset e = f / (2 |grad f / 2|), + outside (G25), with the reciprocals of the semi-axes
    // from the host (nom_q = {1/a, 1/b}) and one reciprocal square root instead of five divisions and a square root: this
    // function is the body of the K*T sequential chain of the nominal rollout, so its dependent-instruction count is its cost
    const float xa = Xabs * p.nom_q[0], yb = Yabs * p.nom_q[1];
    const float f = fmaf(xa, xa, fmaf(yb, yb, -1.0f));
    const float gx = xa * p.nom_q[0], gy = yb * p.nom_q[1];
    const float g2 = fmaf(gx, gx, gy * gy);
    const float e = 0.5f * f * rsqrtf(fmaxf(g2, 1e-24f));   // g floored at 1e-12
    const float over = fmaxf(0.0f, fabsf(e) - p.nom_p[2]);
    const float dv = v - p.nom_p[5];
    return fmaf(p.nom_p[3] * e, e, fmaf(p.nom_p[4] * dv, dv, p.nom_p[6] * over * over));
  }
}

// Terminal cost phi(x_T): w_phi * q_state (G18), or the paper's (23) phi = c4 - c5 s with
// s = distance travelled along the centreline since x_0, wrapped to (-P/2, P/2].
template <int NOM>
__device__ __forceinline__ float terminal_cost(const Params& p, float Xabs, float Yabs, float v, float x0X,
                                               float x0Y) {
  if constexpr (NOM == NOM_RACING) {
    const float P = 4.0f * (p.nom_p[1] + p.nom_p[2] * 1.57079632679489662f + p.nom_p[0]);
    float ds = racing_arclength(p, Xabs, Yabs) - racing_arclength(p, x0X, x0Y);
    if (ds > 0.5f * P) ds -= P;
    if (ds < -0.5f * P) ds += P;
    return fmaf(-p.nom_p[8], ds, p.nom_p[7]);
  } else {
    const float w_phi = (NOM == NOM_GOAL) ? p.nom_p[3] : p.nom_p[7];
    return w_phi * nominal_cost<NOM>(p, Xabs, Yabs, v);
  }
}

// Risk-weighted bilinear costmap lookup between cell centres with clamp-to-edge (G26).
// Layout: the context stores the map as a coefficient grid Q[(H+1)][(W+1)] of float4: with
// (c00, c01, c10, c11) = (c[jy-1][jx-1], c[jy-1][jx], c[jy][jx-1], c[jy][jx]) (indices clamped to the
// map, so clamp-to-edge is baked into the table) and w = risk weight,
//   Q[jy][jx] = w (c00, c01 - c00, c10 - c00, c11 - c10 - c01 + c00)
// so w * bilinear = a + b tx + c ty + d tx ty is one 16-byte load and three FFMA.  Only the coordinate
// is clamped (to [0, W] in the +1-shifted grid).  The grid coordinate is split as (integer bias) +
// (fractional bias + X_rel / res) so the fraction keeps full precision wherever the vehicle is on the
// map.  floor() is taken on the FMA pipe: gx + 1.5*2^23 rounded down has floor(gx) in its low mantissa
// bits (valid for |gx| < 2^22; map sizes are validated), so no F2I/I2F touches the XU pipe.
struct MapFrame {
  float bxf, byf;            // fractional part of (x0 - origin)/res + 1/2
  float lox, hix, loy, hiy;  // clamp bounds of the fractional-frame coordinate
  uint32_t addr_lo, addr_hi; // address of the table entry at index "0 - magic-number bits" (mod 2^32 in the low word): the table lies
                             // inside one 4 GiB window (ra_mppi_create), so an entry's address is addr_hi : (addr_lo + 16 idx), no carry
};

constexpr float kFloorMagic = 12582912.0f;     // 1.5 * 2^23
constexpr uint32_t kFloorMagicBits = 0x4B400000u;

__device__ __forceinline__ MapFrame make_map_frame(const Params& p, float x0X, float x0Y) {
  MapFrame f;
  const float bx = fmaf(x0X - p.map_ox, p.map_inv_res, 0.5f);
  const float by = fmaf(x0Y - p.map_oy, p.map_inv_res, 0.5f);
  const float fx = floorf(bx), fy = floorf(by);
  f.bxf = bx - fx; f.byf = by - fy;
  f.lox = -fx; f.hix = (float)p.map_w - fx;
  f.loy = -fy; f.hiy = (float)p.map_h - fy;
  const uint32_t stride = (uint32_t)(p.map_w + 1);
  // (integer bias y) * (W+1) + (integer bias x), less the magic-number bits the lookup leaves in jx, jy (mod 2^32)
  const uint32_t base = (uint32_t)(int)fy * stride + (uint32_t)(int)fx - ((uint32_t)kFloorMagicBits * stride + (uint32_t)kFloorMagicBits);
  const unsigned long long q0 = reinterpret_cast<unsigned long long>(p.quadmap);
  f.addr_lo = (uint32_t)q0 + (base << 4);
  f.addr_hi = (uint32_t)(q0 >> 32);
  return f;
}

__device__ __forceinline__ float bilinear_weighted(const Params& p, const MapFrame& f, float Xrel, float Yrel) {
  const float gx = fminf(fmaxf(fmaf(Xrel, p.map_inv_res, f.bxf), f.lox), f.hix);
  const float gy = fminf(fmaxf(fmaf(Yrel, p.map_inv_res, f.byf), f.loy), f.hiy);
  const float jx = __fadd_rd(gx, kFloorMagic), jy = __fadd_rd(gy, kFloorMagic);
  const float tx = gx - (jx - kFloorMagic), ty = gy - (jy - kFloorMagic);
  // all index arithmetic is mod 2^32: jy_bits * (W+1) + jx_bits + base is the absolute table index in [0, (H+1)(W+1)), and
  // 16 times it, added to the low address word, cannot carry (the table lies inside one 4 GiB window).  One IMAD + one LEA per
  // lookup; a 64-bit IMAD.WIDE here would hold the FMA pipe for four cycles (profiles/r1c).
  const uint32_t idx = __float_as_uint(jy) * (uint32_t)(p.map_w + 1) + __float_as_uint(jx);
  const float4* addr;
  asm("mov.b64 %0, {%1, %2};" : "=l"(addr) : "r"(f.addr_lo + (idx << 4)), "r"(f.addr_hi));
  RA_DEVICE_CHECK(addr >= p.quadmap && addr < p.quadmap + (size_t)(p.map_h + 1) * (p.map_w + 1));
  const float4 q = __ldg(addr);
  return fmaf(ty, fmaf(tx, q.w, q.z), fmaf(tx, q.y, q.x));
}

}  // namespace ra
