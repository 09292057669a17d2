// philox.cuh -- device Philox4x32-10 and the integer -> normal / uniform maps.
// Counter-based streams as fixed by DESIGN.md readings R1 (layout) and R2 (maps):
//   key = (seed lo32, seed hi32); counter = (c0 = site quad q or 0, c1 = slot, c2 = step t,
//   c3 = stream tag).  One call yields the normals of sites 4q..4q+3.
#pragma once
#include "common.cuh"

namespace phi4 {

struct U4 { uint32_t x, y, z, w; };

__device__ __forceinline__ U4 philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                            uint32_t k0, uint32_t k1) {
  constexpr uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u;
  constexpr uint32_t W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    // one 32x32->64 multiply per product (IMAD.WIDE), one 3-input XOR (LOP3) per word
    const uint64_t p0 = (uint64_t)M0 * (uint64_t)c0;
    const uint64_t p1 = (uint64_t)M1 * (uint64_t)c2;
    c0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
    c2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
    c1 = (uint32_t)p1;
    c3 = (uint32_t)p0;
    k0 += W0;
    k1 += W1;
  }
  return U4{c0, c1, c2, c3};
}

// Round keys k + r * Weyl for r = 0..9, tabulated on the host and passed in kernel-parameter
// space: the per-round XOR then takes its key straight from the constant bank instead of
// spending two integer adds per round per chain.
struct PhiloxKeys { uint32_t k0[10], k1[10]; };

inline PhiloxKeys philox_round_keys(uint64_t seed) {
  PhiloxKeys rk;
  uint32_t a = (uint32_t)seed, b = (uint32_t)(seed >> 32);
  for (int r = 0; r < 10; ++r) { rk.k0[r] = a; rk.k1[r] = b; a += 0x9E3779B9u; b += 0xBB67AE85u; }
  return rk;
}

__device__ __forceinline__ U4 philox4x32_10_rk(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                               const PhiloxKeys& rk) {
  constexpr uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u;
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    const uint64_t p0 = (uint64_t)M0 * (uint64_t)c0;
    const uint64_t p1 = (uint64_t)M1 * (uint64_t)c2;
    c0 = (uint32_t)(p1 >> 32) ^ c1 ^ rk.k0[r];
    c2 = (uint32_t)(p0 >> 32) ^ c3 ^ rk.k1[r];
    c1 = (uint32_t)p1;
    c3 = (uint32_t)p0;
  }
  return U4{c0, c1, c2, c3};
}

__device__ __forceinline__ U4 philox_draw(uint64_t seed, uint32_t tag, uint32_t t, uint32_t slot,
                                          uint32_t q) {
  return philox4x32_10(q, slot, t, tag, (uint32_t)seed, (uint32_t)(seed >> 32));
}

// R2: radius uniform (k+1) 2^-24 in (0,1] (exact in fp32), angle 2 pi k' 2^-24.  Accurate
// logf / sincospif (no fast-math intrinsics); the angle is handed to sincospi as k' 2^-23 so
// that no rounded multiple of pi enters the argument.
__device__ __forceinline__ void box_muller(uint32_t xa, uint32_t xb, float& za, float& zb) {
  float ur = (float)((xa >> 8) + 1u) * 5.9604644775390625e-8f;  // 2^-24
  float r = sqrtf(-2.0f * logf(ur));
  float sn, cs;
  sincospif((float)(xb >> 8) * 1.1920928955078125e-7f, &sn, &cs);  // 2^-23
  za = r * cs;
  zb = r * sn;
}

// Same map on the special-function unit, for the fused mutation kernel whose issue slots the
// normals dominate: lg2.approx on u in (0,1] (absolute error 2^-22 on [0.5,1), 2 ulp below),
// sqrt.approx, sin/cos.approx on the angle reduced exactly (in integers) to [-pi, pi).  The last
// 2^12 radius codes (u > 1 - 2.4e-4, where the absolute error of lg2 would dominate r) take the
// accurate logf.  Resulting |dz| vs the exact map: ~5e-7 typical, < 1e-5 worst case, i.e. a
// proposal perturbation of the order of the fp32 rounding of phi' itself (R2).
__device__ __forceinline__ void box_muller_fast(uint32_t xa, uint32_t xb, float& za, float& zb) {
  const uint32_t m = (xa >> 8) + 1u;                             // 1 .. 2^24
  const float ur = (float)m * 5.9604644775390625e-8f;            // exact
  float w;
  // .ftz forms: every argument here is zero or a normal number (ur >= 2^-24, w >= 0,
  // |th| <= pi), so the subnormal fix-up code of the default forms would never fire
  if (m > 16777216u - 4096u) {
    w = -2.0f * logf(ur);
  } else {
    float l2;
    asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(l2) : "f"(ur));
    w = -1.3862943611198906f * l2;
  }
  float r, cs, sn;
  asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(w));
  const uint32_t kb = xb >> 8;                                   // angle code, 24 bits
  const int sk = (int)kb - (int)((kb & 0x800000u) << 1);         // same angle in [-2^23, 2^23)
  const float th = (float)sk * 3.7450702829238413e-7f;           // 2 pi 2^-24
  asm("cos.approx.ftz.f32 %0, %1;" : "=f"(cs) : "f"(th));
  asm("sin.approx.ftz.f32 %0, %1;" : "=f"(sn) : "f"(th));
  za = r * cs;
  zb = r * sn;
}

__device__ __forceinline__ void normals4_fast(uint64_t seed, uint32_t tag, uint32_t t,
                                              uint32_t slot, uint32_t q, float z[4]) {
  U4 w = philox_draw(seed, tag, t, slot, q);
  box_muller_fast(w.x, w.y, z[0], z[1]);
  box_muller_fast(w.z, w.w, z[2], z[3]);
}

// The four normals of site quad q for (seed, tag, t, slot).
__device__ __forceinline__ void normals4(uint64_t seed, uint32_t tag, uint32_t t, uint32_t slot,
                                         uint32_t q, float z[4]) {
  U4 w = philox_draw(seed, tag, t, slot, q);
  box_muller(w.x, w.y, z[0], z[1]);
  box_muller(w.z, w.w, z[2], z[3]);
}

// R2: accept uniform u = (k+1) 2^-24 from word 0 of the c0 = 0 draw; returns ln u.
__device__ __forceinline__ float log_uniform(uint64_t seed, uint32_t tag, uint32_t t,
                                             uint32_t slot) {
  U4 w = philox_draw(seed, tag, t, slot, 0u);
  return logf((float)((w.x >> 8) + 1u) * 5.9604644775390625e-8f);
}

}  // namespace phi4
