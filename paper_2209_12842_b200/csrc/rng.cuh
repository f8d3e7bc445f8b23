// Counter-based noise in registers: Philox4x32-10 + Box-Muller on exact 23-bit uniforms.
// BASELINE.json fixes the generator; the counter layout is DESIGN.md "RNG layout":
//   ctr = (k, m, call index, stream<<28 | iteration&0x0FFFFFFF),  key = (seed lo, seed hi);
//   EPS stream: call index = t; state-noise streams: the word stream below.
// No [K,M,T,n] noise tensor goes to HBM in fused mode.
#pragma once
#include <cstdint>

#include "ra_params.cuh"

namespace ra {

// One Philox round: two 32x32->64 multiplies (IMAD.WIDE.U32) and two 3-input XORs (LOP3).
__device__ __forceinline__ void philox_round(uint32_t& c0, uint32_t& c1, uint32_t& c2, uint32_t& c3,
                                             uint32_t k0, uint32_t k1) {
  const unsigned long long p0 = (unsigned long long)0xD2511F53u * c0;
  const unsigned long long p1 = (unsigned long long)0xCD9E8D57u * c2;
  const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
  const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
  c1 = (uint32_t)p1;
  c3 = (uint32_t)p0;
  c0 = n0;
  c2 = n2;
}

// rk = the ten (k0,k1) round keys, precomputed on the host because the key is the seed.
__device__ __forceinline__ uint4 philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                               const uint32_t* __restrict__ rk) {
#pragma unroll
  for (int r = 0; r < 10; ++r) philox_round(c0, c1, c2, c3, rk[2 * r], rk[2 * r + 1]);
  return make_uint4(c0, c1, c2, c3);
}

// sin(pi r), cos(pi r) for |r| <= 1/4: minimax-style odd/even polynomials on the FMA pipe.
__device__ __forceinline__ void sincospi_quarter(float r, float& s, float& c) {
  const float r2 = r * r;
  // sin(pi r) = r (pi + r2 (s3 + r2 (s5 + r2 s7)))
  float ps = 0.0821458866f;          //  pi^9/362880
  ps = fmaf(ps, r2, -0.59926452f);   // -pi^7/5040
  ps = fmaf(ps, r2, 2.55016404f);    //  pi^5/120
  ps = fmaf(ps, r2, -5.16771278f);   // -pi^3/6
  const float r3 = r2 * r;
  s = fmaf(r, 3.14159265f, r3 * ps);
  // cos(pi r) = 1 + r2 (c2 + r2 (c4 + r2 (c6 + r2 c8)))
  float pc = 0.235330630f;           //  pi^8/40320
  pc = fmaf(pc, r2, -1.33526277f);   // -pi^6/720
  pc = fmaf(pc, r2, 4.05871213f);    //  pi^4/24
  pc = fmaf(pc, r2, -4.93480220f);   // -pi^2/2
  c = fmaf(pc, r2, 1.0f);
}

// Box-Muller pair from two Philox words.  u1 = ((ra>>9)+1) 2^-23 in (0,1], u2 = (rb>>9) 2^-23
// in [0,1) are exact in fp32, so the transform starts from exact reals.
// The angle 2 pi u2 is reduced exactly in integers: n = rb>>9 in [0,2^23), quadrant q and
// remainder r = u2*2... in [-1/4,1/4] half-turns, then polynomials (no MUFU sin/cos).
__device__ __forceinline__ void box_muller(uint32_t ra, uint32_t rb, float& z0, float& z1) {
  const float u1 = __uint2float_rn((ra >> 9) + 1u) * 1.1920928955078125e-07f;
  const float rho = sqrtf(-2.0f * logf(u1));
  const uint32_t n = rb >> 9;                     // angle = n * 2^-22 half-turns in [0,2)
  const uint32_t q = (n + (1u << 20)) >> 21;      // nearest multiple of 1/2 half-turn, 0..4
  const int rem = (int)n - (int)(q << 21);        // in [-2^20, 2^20]
  const float r = __int2float_rn(rem) * 2.384185791015625e-07f;  // * 2^-22, exact
  float s, c;
  sincospi_quarter(r, s, c);
  // rotate by q quarter-turns
  const float cs = (q & 1u) ? -s : c;
  const float sn = (q & 1u) ? c : s;
  const bool neg = ((q + 0u) & 2u) != 0u;
  z0 = rho * (neg ? -cs : cs);
  z1 = rho * (neg ? -sn : sn);
}

// Fast Box-Muller pair for the state-noise stream (K*M*T*n_x/2 evaluations per iteration): same
// exact uniforms, but log2 / sqrt / sin / cos on the MUFU unit (lg2.approx, sqrt.approx, sin.approx,
// cos.approx).  Error budget: |dz| <= ~2e-6 |z| + 2e-7 / max(rho, 1e-3); scaled by
// sigma_w <= 0.05 that is <= 1e-7 m per step, below the fp32 rounding of the positions themselves.
//   u1 = as_float(0x3F800000 | n1) - (1 - 2^-23) = (n1 + 1) 2^-23      (one funnel shift + one FADD)
//   angle = 2 pi (u2 - 1/2) in [-pi, pi) where MUFU.SIN/COS are most accurate (one funnel shift + one
//   FFMA); the half-turn offset flips both signs.
// Returns the UNSCALED pair (a0, a1) = sqrt(-log2 u1) (cos, sin)(angle); the normals are
// z = -sqrt(2 ln 2) a, and that constant is folded into Params::wscale together with sigma_w, so the
// caller's x += wscale * a is one FFMA per component (12 instructions per pair, 4 of them MUFU).
__device__ __forceinline__ void box_muller_fast(uint32_t ra, uint32_t rb, float& a0, float& a1) {
  const float u1 = __uint_as_float(__funnelshift_r(ra, 0x7Fu, 9)) - 0.99999988079071044921875f;
  float lg, s;
  asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(lg) : "f"(u1));
  asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(s) : "f"(-lg));
  const float th = fmaf(__uint_as_float(__funnelshift_r(rb, 0x7Fu, 9)), 6.283185307179586f, -9.42477796076938f);
  a0 = s * __cosf(th);
  a1 = s * __sinf(th);
}

// Uniform on (-1,1): (2 (r>>9) + 1) 2^-23 - 1, exact.
__device__ __forceinline__ float sym_uniform(uint32_t r) {
  return fmaf(__uint2float_rn(2u * (r >> 9) + 1u), 1.1920928955078125e-07f, -1.0f);
}

// ---- state-noise word stream ------------------------------------------------------
// Realisation (k, m) of a stream owns the word stream  word n = output (n & 3) of Philox4x32-10 at counter
// (k, m, n >> 2, stream<<28 | iteration); step t takes the WD words WD*t .. WD*t + WD - 1 in component order,
// WD = n_x (+ 2 for jump noise: trigger word + one spare so that Box-Muller pairs stay aligned).
// WD = 4: call t.  WD = 8: calls 2t, 2t+1.  WD = 6: 1.5 calls per step -- the rollout kernel walks the horizon in
// pairs of steps and carries the spare half of the middle call (three calls per two steps, not four).
template <int NX, int NOISE> struct NoiseWords { static constexpr int value = NX + (NOISE == NOISE_JUMP ? 2 : 0); };

// The words of step t, on their own (probe, plant, materialised-noise generator, odd last step).
template <int WD>
__device__ __forceinline__ void step_words(const Params& p, uint32_t k, uint32_t m, uint32_t t, uint32_t c3,
                                           uint32_t (&w)[WD]) {
  static_assert(WD == 4 || WD == 6 || WD == 8, "words per step");
  if constexpr (WD == 4) {
    const uint4 a = philox4x32_10(k, m, t, c3, p.rk);
    w[0] = a.x; w[1] = a.y; w[2] = a.z; w[3] = a.w;
  } else if constexpr (WD == 8) {
    const uint4 a = philox4x32_10(k, m, 2u * t, c3, p.rk), b = philox4x32_10(k, m, 2u * t + 1u, c3, p.rk);
    w[0] = a.x; w[1] = a.y; w[2] = a.z; w[3] = a.w; w[4] = b.x; w[5] = b.y; w[6] = b.z; w[7] = b.w;
  } else {
    const uint32_t c = (3u * t) >> 1;   // (6 t) >> 2
    const uint4 a = philox4x32_10(k, m, c, c3, p.rk), b = philox4x32_10(k, m, c + 1u, c3, p.rk);
    const bool odd = (t & 1u) != 0u;    // odd steps start at output 2 of their first call
    w[0] = odd ? a.z : a.x; w[1] = odd ? a.w : a.y; w[2] = odd ? b.x : a.z; w[3] = odd ? b.y : a.w;
    w[4] = odd ? b.z : b.x; w[5] = odd ? b.w : b.y;
  }
}

// The n_x per-step state-noise factors a from the step's words; the additive noise of (6) PAPER.md:63 is
// w_i = Params::wscale[i] * a[i] (wscale = sigma_w times the constant of the noise kind, built by
// ra_mppi_create).
template <int NX, int NOISE>
__device__ __forceinline__ void noise_from_words(const Params& p, const uint32_t (&w)[NoiseWords<NX, NOISE>::value],
                                                 float (&z)[NX]) {
#pragma unroll
  for (int i = 0; i < NX; i += 2) {
    if constexpr (NOISE == NOISE_UNIFORM) { z[i] = sym_uniform(w[i]); z[i + 1] = sym_uniform(w[i + 1]); }
    else box_muller_fast(w[i], w[i + 1], z[i], z[i + 1]);
  }
  if constexpr (NOISE == NOISE_JUMP) {
    // jump of unit length in a uniformly random direction z/|z| (the common factor of the Gaussian
    // draws cancels; its sign is in wscale), with probability noise_p[0]  (G29)
    const float uj = __uint2float_rn(w[NX] >> 9) * 1.1920928955078125e-07f;
    float n2 = 0.0f;
#pragma unroll
    for (int i = 0; i < NX; ++i) n2 = fmaf(z[i], z[i], n2);
    const bool jump = (uj < p.noise_p[0]) && (n2 > 0.0f);
    const float inv = jump ? rsqrtf(n2) : 0.0f;
#pragma unroll
    for (int i = 0; i < NX; ++i) z[i] *= inv;
  }
}

template <int NX, int NOISE>
__device__ __forceinline__ void state_noise(const Params& p, uint32_t k, uint32_t m, uint32_t t,
                                            uint32_t c3, float (&z)[NX]) {
  uint32_t w[NoiseWords<NX, NOISE>::value];
  step_words(p, k, m, t, c3, w);
  noise_from_words<NX, NOISE>(p, w, z);
}

}  // namespace ra
