// Steps A2-A5 of one scatterer: geometry -> (gate, Doppler bin, gate weight, phase) ->
// complex amplitude.  Paper: `scatterers_range`, `scatterers_complex_amplitudes`, the coordinates of
// `rasterize`.  Used by every accumulation kernel and by the index-only kernel.
#pragma once
#include <climits>

#include "sim_internal.h"

namespace simk {

// 1.5 * 2^(52 - kFracBits): adding it to v (|v| < 2^11) leaves floor/round(v * 2^20) in the low word.
constexpr double kMagicFx = 6442450944.0;        // 1.5 * 2^32
constexpr double kMagicFxHalf = 6442450944.5;    // the same + 0.5 (nearest-bin rule, ties up)
constexpr double kMagicPhase = 402653184.0;      // 1.5 * 2^28: low word = round(q * 2^24)
constexpr int kFxOne = 1 << kFracBits;

// index routines: the canonical fp64 sequence for every scatterer, or a polynomial path (analytic Doppler /
// pulse-pair Doppler) with the canonical sequence inside the guard band
enum { kIdxCanonical = 0, kIdxFast = 1, kIdxFastPulsePair = 2 };

// What the index part of one scatterer yields.
struct Idx {
  int g0;      // gate of the lower half, in [-1, G-1]
  int k;       // Doppler bin, UNWRAPPED: congruent to the bin mod N, |k| < 2^30
  float w1;    // weight of gate g0+1 (gate g0 gets 1 - w1)
  float fr;    // frac(2R/lambda) mapped to [-0.5, 0.5) cycles
  float gfx;   // gf * 2^kFracBits as a float (for 1/R^2)
};

// frac(q) of q cycles as a float in [-0.5, 0.5): round(q * 2^24) sits in the low word after the magic add
__device__ __forceinline__ float cycles_fraction(double q) {
  const int lo = __double2loint(__dadd_rn(q, kMagicPhase));
  return (float)(int)((unsigned)lo << 8) * 2.3283064365386963e-10f;  // * 2^-32
}

// ---------------------------------------------------------------------------------------------
// CANONICAL fp64 INDEX SEQUENCE of DESIGN.md, from dx, dy, dz.  Explicit round-to-nearest
// intrinsics: nvcc must not contract a*b+c differently from the definition.  Out of line (the fast
// path calls it only inside the guard band) and fed by value.
// Returns (g0, k unwrapped, bits of w1, bits of fr); g0 = SIM_GATE_NONE when the scatterer is dropped.
// ---------------------------------------------------------------------------------------------
struct CanonConsts {
  double rg0, inv_dR, cD, two_over_lambda, fr0, svx, svy, svz, pri, cP;
  int G, N, mode;
};

static __device__ __noinline__ int4 canonical_tail(CanonConsts c, double dx, double dy, double dz, float vxf,
                                                   float vyf, float vzf) {
  const int4 dropped = make_int4(SIM_GATE_NONE, -1, 0, 0);
  const double R2 = __fma_rn(dz, dz, __fma_rn(dy, dy, __dmul_rn(dx, dx)));
  const double R = __dsqrt_rn(R2);
  const double delta = __dsub_rn(R, c.rg0);
  const double gf = __dmul_rn(delta, c.inv_dR);
  if (!(gf >= -1.0 && gf < (double)c.G)) return dropped;  // touches no gate (NaN lands here too)
  const double g0d = floor(gf);
  const double dvx = __dsub_rn((double)vxf, c.svx);
  const double dvy = __dsub_rn((double)vyf, c.svy);
  const double dvz = __dsub_rn((double)vzf, c.svz);
  double kf;
  if (c.mode == SIM_DOPPLER_PULSE_PAIR) {
    // Algorithm 1 lines 5-7: the offset one PRI later, R' - R, in bins (reading R4)
    const double dx1 = __fma_rn(dvx, c.pri, dx), dy1 = __fma_rn(dvy, c.pri, dy), dz1 = __fma_rn(dvz, c.pri, dz);
    const double R1 = __dsqrt_rn(__fma_rn(dz1, dz1, __fma_rn(dy1, dy1, __dmul_rn(dx1, dx1))));
    kf = __dmul_rn(__dsub_rn(R1, R), c.cP);
  } else {
    const double rdot = __ddiv_rn(__fma_rn(dvz, dz, __fma_rn(dvy, dy, __dmul_rn(dvx, dx))), R);
    kf = __dmul_rn(rdot, c.cD);
  }
  if (!(fabs(kf) < 1073741824.0)) return dropped;
  const double kk = floor(__dadd_rn(kf, 0.5));
  // the bin is returned UNWRAPPED (|kk| < 2^30), like the polynomial path's: whoever needs the bin takes it mod N
  const double q = __fma_rn(delta, c.two_over_lambda, c.fr0);  // only the fraction of 2R/lambda matters
  return make_int4((int)g0d, (int)kk, __float_as_int((float)__dsub_rn(gf, g0d)),
                   __float_as_int(cycles_fraction(q)));
}

__device__ __forceinline__ bool canonical(const AccParams& p, double dx, double dy, double dz, float vxf,
                                          float vyf, float vzf, Idx& o) {
  CanonConsts c;
  c.rg0 = p.rg0; c.inv_dR = p.inv_dR; c.cD = p.cD; c.two_over_lambda = p.two_over_lambda; c.fr0 = p.fr0;
  c.svx = p.svx; c.svy = p.svy; c.svz = p.svz; c.G = p.G; c.N = p.N;
  c.pri = p.pri; c.cP = p.cP; c.mode = p.doppler_mode;
  const int4 r = canonical_tail(c, dx, dy, dz, vxf, vyf, vzf);
  if (r.x == SIM_GATE_NONE) return false;
  o.g0 = r.x;
  o.k = r.y;
  o.w1 = __int_as_float(r.z);
  o.fr = __int_as_float(r.w);
  o.gfx = ((float)r.x + o.w1) * (float)kFxOne;
  return true;
}

// Steps A2-A4 in two parts, so that a warp whose scatterers all miss the window can stop after the first.
//   MODE = kIdxCanonical: the canonical sequence for every scatterer.
//   MODE = kIdxFast, kIdxFastPulsePair:  everything is a short polynomial in u = R^2 - rg0^2 (no sqrt, no divide):
//       gf = (R - rg0)/dR = u (g1 + u (g2 + u g3)),   kf = num cD / R = num (j0 + u (j1 + u j2)),
//     gate and bin are read from 2^-20 fixed point; whenever a coordinate lies within `guard` of an
//     integer boundary the canonical sequence decides (bit-exact indices).
struct Pre {
  double dx, dy, dz, u;
};

// Offsets from the satellite and the window pre-test.  `live` in: the scatterer is a candidate (s0dA > 0);
// out: it may land in the gate window.
template <int MODE>
__device__ __forceinline__ Pre pre_part(const AccParams& p, float xf, float yf, float zf, bool& live) {
  Pre q;
  q.dx = __dsub_rn((double)xf, p.sx);
  q.dy = __dsub_rn((double)yf, p.sy);
  q.dz = __dsub_rn((double)zf, p.sz);
  q.u = 0.0;
  if (MODE != kIdxCanonical) {
    // the three squares cancel against -rg0^2; every rounding is <= ulp(rg0^2) ~ 1e-4 m^2 (<< guard)
    q.u = fma(q.dz, q.dz, fma(q.dy, q.dy, fma(q.dx, q.dx, p.neg_rg0sq)));
    live = live && (q.u >= p.uw_lo) && (q.u <= p.uw_hi);   // false: certainly outside the window (or NaN)
  }
  return q;
}

// The polynomial index path (MODE = kIdxFast or kIdxFastPulsePair) in the form the production kernel keeps alive across the amplitude code: the two fixed-point
// coordinates and the phase; gate, bin, weight and the guard-band test are derived from them afterwards.
struct Fx {
  int gfx;     // floor(gf * 2^kFracBits)
  int kfx;     // floor((kf + 0.5) * 2^kFracBits); INT_MIN when |kf| >= 1024 (the fixed-point read would be meaningless)
  float fr;    // frac(2R/lambda) mapped to [-0.5, 0.5) cycles, in units of 2^-32 cycles
};
constexpr float kFrUnit = 2.3283064365386963e-10f;   // 2^-32: Fx::fr -> cycles

template <int MODE>
__device__ __forceinline__ Fx index_fx(const AccParams& p, const Pre& q, float xf, float yf, float zf, float vxf, float vyf,
                                       float vzf) {
  Fx o;
  const double u = q.u;
  const double gf = u * fma(u, fma(u, p.g3, p.g2), p.g1);
  o.gfx = __double2loint(__dadd_rd(gf, kMagicFx));
  const double dvx = (double)vxf - p.svx, dvy = (double)vyf - p.svy, dvz = (double)vzf - p.svz;
  const double num = fma(dvz, q.dz, fma(dvy, q.dy, dvx * q.dx));
  double kf;
  if (MODE == kIdxFastPulsePair) {
    const double dv2 = fma(dvz, dvz, fma(dvy, dvy, dvx * dvx));
    const double w = p.pri * fma(dv2, p.pri, num + num);
    const double e = fma(w, p.inv_2rg0, gf * p.two_dR) * p.inv_2rg0;
    kf = (w * p.cP_2rg0) * fma(e, e - 1.0, 1.0);
  } else {
    kf = num * fma(u, fma(u, p.j2, p.j1), p.j0);
  }
  const int kfx = __double2loint(__dadd_rd(kf, kMagicFxHalf));
  o.kfx = (fabs(kf) < 1024.0) ? kfx : INT_MIN;
  // frac(2R/lambda) in units of 2^-32 cycles (two's complement wrap = the fraction in [-1/2, 1/2)): the magic number
  // rides in the addend (fr0m = fr0 + 1.5 * 2^28, rounded to 2^-24 cycles)
  o.fr = (float)(int)((unsigned)__double2loint(fma(gf, p.cq, p.fr0m)) << 8);
  return o;
}

template <int MODE>
__device__ __forceinline__ int fx_bin(const AccParams& p, const Fx& f) {
  return f.kfx >> kFracBits;
}

// True when a coordinate lies inside the guard band (or the Doppler coordinate was out of the fixed-point range): the
// canonical sequence has to decide.
template <int MODE>
__device__ __forceinline__ bool fx_near(const AccParams& p, const Fx& f) {
  const int gk = MODE == kIdxFastPulsePair ? p.guard_k : p.guard;   // pulse-pair: wider Doppler guard band
  const unsigned span = (unsigned)(kFxOne - 2 * p.guard), span_k = (unsigned)(kFxOne - 2 * gk);
  const int gfrac = f.gfx & (kFxOne - 1), kfrac = f.kfx & (kFxOne - 1);
  return ((unsigned)(gfrac - p.guard) >= span) | ((unsigned)(kfrac - gk) >= span_k) | (f.kfx == INT_MIN);
}

__device__ __forceinline__ float sqrt_approx(float v) {
  float r;
  asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(v));
  return r;
}
__device__ __forceinline__ float ex2_approx(float v) {
  float r;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(v));
  return r;
}

// Tabulated antenna pattern (reading R9): complex gain at the direction cosines (u, v) by bilinear
// interpolation in p.lut [nv][nu]; false outside the recorded grid.  fp32; the four nodes come through the read-only
// path (the table is small and shared by every scatterer: L1/L2 resident).
__device__ __forceinline__ bool lut_gain(const AccParams& p, float u, float v, float2& g) {
  const float fu = (u - p.lut_u0) * p.lut_inv_du, fv = (v - p.lut_v0) * p.lut_inv_dv;
  if (!(fu >= 0.0f && fu <= (float)(p.lut_nu - 1) && fv >= 0.0f && fv <= (float)(p.lut_nv - 1))) return false;
  const int i = min((int)fu, p.lut_nu - 2), j = min((int)fv, p.lut_nv - 2);   // the last node belongs to the last cell
  const float a = fu - (float)i, b = fv - (float)j;
  const float2* t = p.lut + (size_t)j * p.lut_nu + i;
  const float2 t00 = __ldg(t), t01 = __ldg(t + 1), t10 = __ldg(t + p.lut_nu), t11 = __ldg(t + p.lut_nu + 1);
  const float w00 = (1.0f - a) * (1.0f - b), w01 = a * (1.0f - b), w10 = (1.0f - a) * b, w11 = a * b;
  g.x = fmaf(w11, t11.x, fmaf(w10, t10.x, fmaf(w01, t01.x, w00 * t00.x)));
  g.y = fmaf(w11, t11.y, fmaf(w10, t10.y, fmaf(w01, t01.y, w00 * t00.y)));
  return true;
}

// Step A5: sqrt(s0dA) G / R^2 exp(-i 2 pi fr), all fp32.  Returns an upper bound of |c| (within sqrt 2) in A.
//   1/R^2 from the gate coordinate; offsets d from the satellite in fp32 (hi + lo split only where it matters: z);
//   (e1, e2, boresight) orthonormal, e1 along track (reading R9): analytic gain exp(-alpha sin^2(theta)) with
//   sin^2(theta) = ((d.e1)^2 + (d.e2)^2) / R^2, or the tabulated complex gain at (u, v) = (d.e1, d.e2) / R.
template <bool LUT>
__device__ __forceinline__ float2 amplitude_t(const AccParams& p, float xf, float yf, float zf, float gfx,
                                              float fr, float s0dA, float& A) {
  const float dx = xf - p.sxh, dy = yf - p.syh, dz = (zf - p.szh) - p.szl;
  const float inv_R2 = fmaf(gfx, fmaf(gfx, p.a2, p.a1), p.a0);
  const float p1 = fmaf(dz, p.e1z, fmaf(dy, p.e1y, dx * p.e1x));
  const float p2 = fmaf(dz, p.e2z, fmaf(dy, p.e2y, dx * p.e2x));
  float sn, cs;
  __sincosf(6.283185307179586f * fr, &sn, &cs);
  if (LUT) {
    const float inv_R = sqrt_approx(inv_R2);
    float2 g;
    if (!lut_gain(p, p1 * inv_R, p2 * inv_R, g)) {
      A = 0.0f;
      return make_float2(0.0f, 0.0f);
    }
    const float A0 = sqrt_approx(s0dA) * inv_R2;
    A = A0 * (fabsf(g.x) + fabsf(g.y));
    const float gr = A0 * g.x, gi = A0 * g.y;
    return make_float2(fmaf(gr, cs, gi * sn), fmaf(gi, cs, -gr * sn));   // (gr + i gi)(cs - i sn)
  }
  const float t = fmaf(p2, p2, p1 * p1);
  A = sqrt_approx(s0dA) * ex2_approx(t * (inv_R2 * p.neg_alpha_log2e)) * inv_R2;
  return make_float2(A * cs, -A * sn);
}
// ---- packed fp32 pairs (sm_100: one instruction, two lanes of data): two scatterers at a time ----
__device__ __forceinline__ unsigned long long pk(float2 a) {
  unsigned long long r;
  asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(a.x), "f"(a.y));
  return r;
}
__device__ __forceinline__ float2 upk(unsigned long long r) {
  float2 a;
  asm("mov.b64 {%0, %1}, %2;" : "=f"(a.x), "=f"(a.y) : "l"(r));
  return a;
}
__device__ __forceinline__ float2 fma2(float2 a, float2 b, float2 c) {
  unsigned long long d;
  asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(pk(a)), "l"(pk(b)), "l"(pk(c)));
  return upk(d);
}
__device__ __forceinline__ float2 mul2(float2 a, float2 b) {
  unsigned long long d;
  asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(pk(a)), "l"(pk(b)));
  return upk(d);
}
__device__ __forceinline__ float2 bc(float s) { return make_float2(s, s); }

// Step A5 for TWO scatterers (components .x and .y of every argument), analytic gain: the same arithmetic as
// amplitude_t<false>, with d.e1 and d.e2 taken straight from the coordinates (e1c = -r_sat.e1, e2c = -r_sat.e2 are host
// constants) and the phase given in units of 2^-32 cycles (Fx::fr).  cre, cim: real and imaginary parts of the two amplitudes.
__device__ __forceinline__ void amplitude_pair(const AccParams& p, float2 x, float2 y, float2 z, float2 gfx, float2 fr,
                                               float2 s0dA, float2& A, float2& cre, float2& cim) {
  const float2 inv_R2 = fma2(gfx, fma2(gfx, bc(p.a2), bc(p.a1)), bc(p.a0));
  const float2 p1 = fma2(z, bc(p.e1z), fma2(y, bc(p.e1y), fma2(x, bc(p.e1x), bc(p.e1c))));
  const float2 p2 = fma2(z, bc(p.e2z), fma2(y, bc(p.e2y), fma2(x, bc(p.e2x), bc(p.e2c))));
  const float2 t = fma2(p2, p2, mul2(p1, p1));
  const float2 arg = mul2(t, mul2(inv_R2, bc(p.neg_alpha_log2e)));
  const float2 g = make_float2(sqrt_approx(s0dA.x) * ex2_approx(arg.x), sqrt_approx(s0dA.y) * ex2_approx(arg.y));
  A = mul2(g, inv_R2);
  const float2 ph = mul2(fr, bc(-6.283185307179586f * kFrUnit));   // -2 pi frac(2R/lambda)
  float2 sn, cs;
  __sincosf(ph.x, &sn.x, &cs.x);
  __sincosf(ph.y, &sn.y, &cs.y);
  cre = mul2(A, cs);
  cim = mul2(A, sn);
}

// run-time choice (kernels off the hot path: reference, regular mode)
__device__ __forceinline__ float2 amplitude(const AccParams& p, float xf, float yf, float zf, float gfx, float fr,
                                            float s0dA, float& A) {
  return p.lut != nullptr ? amplitude_t<true>(p, xf, yf, zf, gfx, fr, s0dA, A) : amplitude_t<false>(p, xf, yf, zf, gfx, fr, s0dA, A);
}

}  // namespace simk
