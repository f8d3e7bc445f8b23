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

// Box-Muller pair for the state-noise streams (K*M*T*n_x/2 evaluations per iteration) from ONE Philox word
// (DESIGN.md "RNG layout"): radius uniform u1 = ((w & 0xFFFF) + 1/2) 2^-16 in (0,1), angle uniform u2 = (w >> 9) 2^-23
// in [0,1), both exact in fp32; log2 / sqrt / sin / cos on the MUFU unit (lg2.approx, sqrt.approx, sin.approx,
// cos.approx).  Error budget: |dz| <= ~2e-6 |z| + 2e-7 / max(rho, 1e-3); scaled by
// sigma_w <= 0.05 that is <= 1e-7 m per step, below the fp32 rounding of the positions themselves.
//   u1: PRMT builds the float 1 + lo 2^-23 (bytes 0x3F80 : lo16), one FFMA scales it: (1 + lo 2^-23) 128 - (128 - 2^-17)
//       = (lo + 1/2) 2^-16 exactly (only relative accuracy matters under the logarithm).
//   angle = 2 pi (u2 - 1/2) in [-pi, pi) where MUFU.SIN/COS are most accurate: one funnel shift drops the top 23 bits
//       of the word into the mantissa of x = 1 + u2 in [1,2), one FFMA forms 2 pi x - 3 pi (the cancellation is against
//       2 pi, so the angle is good to 5e-7 rad).  The half-turn offset flips both signs.
// Returns the UNSCALED pair (a0, a1) = sqrt(-log2 u1) (cos, sin)(angle); the normals are z = -sqrt(2 ln 2) a, and
// that constant is folded into Params::wscale together with sigma_w, so the caller's x += wscale * a is one FFMA
// per component.  12 instructions per pair: 2 on the ALU pipe, 6 on the FMA pipe, 4 MUFU.
__device__ __forceinline__ void box_muller16_fast(uint32_t w, float& a0, float& a1) {
  const float u1 = fmaf(__uint_as_float(__byte_perm(w, 0x3F800000u, 0x7610)), 128.0f, -127.99999237060546875f);
  float lg, s;
  asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(lg) : "f"(u1));
  asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(s) : "f"(-lg));
  const float th = fmaf(__uint_as_float(__funnelshift_r(w, 0x7Fu, 9)), 6.283185307179586f, -9.42477796076938f);
  a0 = s * __cosf(th);
  a1 = s * __sinf(th);
}

// h 2^-16 for a 16-bit field already placed in the low mantissa bits (bits 0x3F80 : h = 1 + h 2^-23), exact
__device__ __forceinline__ float unit16(uint32_t bits) { return fmaf(__uint_as_float(bits), 128.0f, -128.0f); }

// Two uniforms on (-1,1) from one word: (2 h + 1) 2^-16 - 1 for the high and the low half, exact (h 2^-15 by one FFMA,
// then one FADD; no I2F on the XU pipe).
__device__ __forceinline__ void sym_uniform16(uint32_t w, float& z_hi, float& z_lo) {
  const float th = fmaf(__uint_as_float(__byte_perm(w, 0x3F800000u, 0x7632)), 256.0f, -256.0f);
  const float tl = fmaf(__uint_as_float(__byte_perm(w, 0x3F800000u, 0x7610)), 256.0f, -256.0f);
  z_hi = th - 0.9999847412109375f;   // 1 - 2^-16
  z_lo = tl - 0.9999847412109375f;
}

// ---- state-noise word stream ------------------------------------------------------
// Realisation (k, m) of a stream owns the word stream  word n = output (n & 3) of Philox4x32-10 at counter
// (k, m, n >> 2, stream<<28 | iteration); step t takes the WD words WD*t .. WD*t + WD - 1, word j -> state
// components (2j, 2j+1); WD = n_x / 2 (+ 1 for jump noise: a word whose high half is the trigger).
// WD = 2: one call per two steps.  WD = 3: three calls per four steps.  WD = 4: one call per step.  The rollout
// kernel walks the horizon in groups of steps that share calls and carries the spare words.
template <int NX, int NOISE> struct NoiseWords { static constexpr int value = NX / 2 + (NOISE == NOISE_JUMP ? 1 : 0); };

// The words of step t, on their own (probe, plant, materialised-noise generator, ragged last steps).
template <int WD>
__device__ __forceinline__ void step_words(const Params& p, uint32_t k, uint32_t m, uint32_t t, uint32_t c3,
                                           uint32_t (&w)[WD]) {
  static_assert(WD == 2 || WD == 3 || WD == 4, "words per step");
  if constexpr (WD == 4) {
    const uint4 a = philox4x32_10(k, m, t, c3, p.rk);
    w[0] = a.x; w[1] = a.y; w[2] = a.z; w[3] = a.w;
  } else if constexpr (WD == 2) {
    const uint4 a = philox4x32_10(k, m, t >> 1, c3, p.rk);
    const bool odd = (t & 1u) != 0u;
    w[0] = odd ? a.z : a.x; w[1] = odd ? a.w : a.y;
  } else {
    const uint32_t n0 = 3u * t, c = n0 >> 2, o = n0 & 3u;   // first word = output o of call c
    const uint4 a = philox4x32_10(k, m, c, c3, p.rk);
    const uint32_t av[4] = {a.x, a.y, a.z, a.w};
    uint32_t bv[4] = {0u, 0u, 0u, 0u};
    if (o >= 2u) {   // the step runs over into the next call
      const uint4 b = philox4x32_10(k, m, c + 1u, c3, p.rk);
      bv[0] = b.x; bv[1] = b.y; bv[2] = b.z; bv[3] = b.w;
    }
#pragma unroll
    for (int i = 0; i < 3; ++i) {
      const uint32_t n = o + (uint32_t)i;
      uint32_t v = 0u;
#pragma unroll
      for (int j = 0; j < 4; ++j) v = (n == (uint32_t)j) ? av[j] : ((n == (uint32_t)(j + 4)) ? bv[j] : v);
      w[i] = v;
    }
  }
}

// The n_x per-step state-noise factors a from the step's words; the additive noise of (6) PAPER.md:63 is
// w_i = Params::wscale[i] * a[i] (wscale = sigma_w times the constant of the noise kind, built by
// ra_mppi_create).
template <int NX, int NOISE>
__device__ __forceinline__ void noise_from_words(const Params& p, const uint32_t (&w)[NoiseWords<NX, NOISE>::value],
                                                 float (&z)[NX]) {
#pragma unroll
  for (int j = 0; j < NX / 2; ++j) {
    if constexpr (NOISE == NOISE_UNIFORM) sym_uniform16(w[j], z[2 * j], z[2 * j + 1]);
    else box_muller16_fast(w[j], z[2 * j], z[2 * j + 1]);
  }
  if constexpr (NOISE == NOISE_JUMP) {
    // jump of unit length in a uniformly random direction z/|z| (the common factor of the Gaussian
    // draws cancels; its sign is in wscale), with probability noise_p[0]  (G29)
    const float uj = unit16(__byte_perm(w[NX / 2], 0x3F800000u, 0x7632));
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
