// REGULAR MODE (reading R5): the surface is updated at every
// pulse and the raw data of a pulse are the complex sum of all scatterers per range gate.  Scatterers and
// satellite in uniform motion from the states given at pulse 0:
//     Y[j][g] = sum_p w_g(R_p(t_j)) sqrt(s0dA_p) G(theta_p(t_j)) / R_p(t_j)^2 exp(-i 4 pi R_p(t_j) / lambda),  t_j = j / PRF.
// Work = scatterers x pulses.  No Doppler axis, no FFT: this is the at-scale truth the fast mode approximates.
//
// One WARP = one SCATTERER at a time, its 32 LANES = the 32 PULSES of the block's pulse tile; a block = 16 warps x one
// slice of the scatterers, with a shared-memory tile Y[32 pulses][G].  Lanes of a warp always hit different rows
// (pulses), so the adds of a warp never replay; warps meet in a cell only when two scatterers fall into the same gate
// at the same pulse.  The tile is block floating point like the accumulation kernel's: native int32 reductions of
// round(w c s), s a power of two per epoch of 8192 scatterers (<= 8192 adds of <= 2^17 per cell: no overflow),
// brighter contributions to an exact global fp32 reduction, tile flushed (x 1/s) into Y at every epoch end.
// The block's threads first turn a chunk of scatterers into per-scatterer constants (u(t) = R(t)^2 - rg0^2 =
// u0 + a t + b t^2 in fp64, antenna projections linear in t; raw inputs of the next chunk prefetched into
// registers), then every warp walks its share of the chunk (shared-memory broadcasts).
// Per (scatterer, pulse): 2 DFMA for u, the gate coordinate by the same polynomial as the fast-mode index path,
// phase fraction in fp64, the rest in fp32.
#include "scatter_math.cuh"

namespace simk {

constexpr int kRegWarps = 16;                  // warps per block
constexpr int kRegThreads = kRegWarps * 32;
constexpr int kRegChunk = kRegThreads;         // scatterers per shared-memory chunk: one per thread to prepare
constexpr int kRegJT = 32;                     // pulses per block = lanes of a warp
constexpr int kRegEpochChunks = 16;            // chunks per fixed-point epoch: 8192 scatterers, <= 8192 adds per cell
constexpr int kRegCap = 17;                    // admitted |c| s <= 2^17: 8192 adds (+ rounding) stay below 2^31
constexpr int kRegTarget = 15;                 // gmean(sqrt(s0dA) / rg0^2) s in [2^15, 2^16)

struct RegParams {
  AccParams a;       // geometry constants (make_acc_params)
  float2* Y;         // [n_pulses][G]
  long long j0;      // first pulse, relative to the instant of the satellite state
  int n_pulses;      // pulses of the call
  int n_slices;      // scatterer slices (gridDim.y)
  double prf;        // t_j = j / PRF, the oracle's expression
};

size_t regular_smem_bytes(int G) {
  return (size_t)kRegJT * (2 * G + 1) * sizeof(float) + (size_t)kRegChunk * (3 * sizeof(double) + 6 * sizeof(float));
}

__global__ void __launch_bounds__(kRegThreads) regular_kernel(RegParams rp) {
  const AccParams& p = rp.a;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int G = p.G, LD = 2 * G + 1;
  double* s_u0 = reinterpret_cast<double*>(smem_raw);   // [chunk] u at pulse 0
  double* s_a = s_u0 + kRegChunk;                        // [chunk] 2 d.dv
  double* s_b = s_a + kRegChunk;                         // [chunk] |dv|^2
  float* s_p1 = reinterpret_cast<float*>(s_b + kRegChunk);   // [chunk] d.e1, then dv.e1, d.e2, dv.e2, sqrt(s0dA)
  float* s_p1v = s_p1 + kRegChunk;
  float* s_p2 = s_p1v + kRegChunk;
  float* s_p2v = s_p2 + kRegChunk;
  float* s_amp = s_p2v + kRegChunk;
  float* s_pad = s_amp + kRegChunk;                      // (unused sixth array keeps the tile 8-byte aligned)
  float* tile = s_pad + kRegChunk;                       // [32 pulses][2G+1]: re, im interleaved per gate
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  int* itile = reinterpret_cast<int*>(tile);             // block floating point: round(w c s), s = 2^s_ex per epoch
  __shared__ int s_ex, s_have;
  for (int i = tid; i < kRegJT * LD; i += kRegThreads) itile[i] = 0;
  if (tid == 0) s_have = 0;
  const unsigned row_a = (unsigned)__cvta_generic_to_shared(itile + (size_t)lane * LD);

  const long long j = rp.j0 + (long long)blockIdx.x * kRegJT + lane;
  const bool pulse_ok = (long long)blockIdx.x * kRegJT + lane < rp.n_pulses;
  const double t = __ddiv_rn((double)j, rp.prf);
  const float tf = (float)t;

  const unsigned long long per = (p.n + rp.n_slices - 1) / rp.n_slices;
  const unsigned long long lo = per * blockIdx.y, hi = (lo + per < p.n) ? lo + per : p.n;
  float in[7];
  auto fetch = [&](unsigned long long base) {   // this thread's scatterer of the chunk at `base`, raw
    const unsigned long long q = base + tid;
    const bool v = q < hi;
    in[0] = v ? p.x[q] : 0.0f; in[1] = v ? p.y[q] : 0.0f; in[2] = v ? p.z[q] : 0.0f;
    in[3] = v ? p.vx[q] : 0.0f; in[4] = v ? p.vy[q] : 0.0f; in[5] = v ? p.vz[q] : 0.0f;
    in[6] = v ? p.s0dA[q] : 0.0f;
  };
  const int rows = min(kRegJT, rp.n_pulses - blockIdx.x * kRegJT);
  auto flush = [&]() {   // tile -> Y (x 1/s), tile zeroed; gate fastest across threads
    __syncthreads();
    if (s_have) {
      const float inv_s = __int_as_float((127 - s_ex) << 23);
      for (int e = tid; e < rows * G; e += kRegThreads) {
        const int r = e / G, g = e - r * G;
        int* c = itile + (size_t)r * LD + 2 * g;
        const int re = c[0], im = c[1];
        if (re | im) {
          c[0] = 0;
          c[1] = 0;
          atomicAdd(&rp.Y[((size_t)blockIdx.x * kRegJT + r) * G + g], make_float2((float)re * inv_s, (float)im * inv_s));
        }
      }
    }
    __syncthreads();
    if (tid == 0) s_have = 0;
  };
  if (lo < hi) fetch(lo);
  int chunk_in_epoch = 0;
  for (unsigned long long base = lo; base < hi; base += kRegChunk) {
    if (chunk_in_epoch == kRegEpochChunks) {
      flush();
      chunk_in_epoch = 0;
    }
    ++chunk_in_epoch;
    const int m = (int)((hi - base < (unsigned long long)kRegChunk) ? hi - base : kRegChunk);
    __syncthreads();   // the previous chunk has been consumed (and, the first time, the tile is zero)
    const int have0 = s_have;   // read between two barriers with no writer in between: block-uniform
    if (tid < m) {
      const int i = tid;
      const float s0 = in[6];
      const double dx = __dsub_rn((double)in[0], p.sx), dy = __dsub_rn((double)in[1], p.sy), dz = __dsub_rn((double)in[2], p.sz);
      const double dvx = (double)in[3] - p.svx, dvy = (double)in[4] - p.svy, dvz = (double)in[5] - p.svz;
      s_u0[i] = fma(dz, dz, fma(dy, dy, fma(dx, dx, p.neg_rg0sq)));
      s_a[i] = 2.0 * fma(dvz, dz, fma(dvy, dy, dvx * dx));
      s_b[i] = fma(dvz, dvz, fma(dvy, dvy, dvx * dvx));
      s_p1[i] = (float)(dx * (double)p.e1x + dy * (double)p.e1y + dz * (double)p.e1z);
      s_p1v[i] = (float)(dvx * (double)p.e1x + dvy * (double)p.e1y + dvz * (double)p.e1z);
      s_p2[i] = (float)(dx * (double)p.e2x + dy * (double)p.e2y + dz * (double)p.e2z);
      s_p2v[i] = (float)(dvx * (double)p.e2x + dvy * (double)p.e2y + dvz * (double)p.e2z);
      s_amp[i] = (s0 > 0.0f) ? sqrt_approx(s0) : 0.0f;   // s0dA <= 0 or NaN: contributes nothing
    }
    __syncthreads();
    if (!have0) {   // the first chunk of the epoch with live scatterers fixes the epoch's scale
      if (warp == 0) {
        int cnt = 0, slog = 0;
        for (int i = lane; i < m; i += 32) {
          const float a = s_amp[i] * p.a0;   // the amplitude at full antenna gain
          if (a > 0.0f) {
            ++cnt;
            slog += __float_as_int(a) >> 16;   // log2, 2^-7 units
          }
        }
        cnt = __reduce_add_sync(0xffffffffu, cnt);
        slog = __reduce_add_sync(0xffffffffu, slog);
        if (lane == 0 && cnt > 0) {
          const int E = (slog / cnt) >> 7;   // biased exponent of the geometric mean
          s_ex = max(-100, min(120, kRegTarget - (E - 127)));
          s_have = 1;
        }
      }
      __syncthreads();
    }
    if (base + kRegChunk < hi) fetch(base + kRegChunk);   // in flight during the evaluation below
    if (!pulse_ok || !s_have) continue;
    const float sc = __int_as_float((s_ex + 127) << 23);
    const int hi_bits = (kRegCap - s_ex + 127) << 23;   // bits of 2^cap / s
#pragma unroll 2
    for (int i = warp; i < m; i += kRegWarps) {   // warp-uniform: every lane reads the same scatterer (broadcast)
      const float amp = s_amp[i];
      if (!(amp > 0.0f)) continue;
      const double u = fma(t, fma(t, s_b[i], s_a[i]), s_u0[i]);
      if (!(u >= p.uw_lo && u <= p.uw_hi)) continue;              // outside the window at this pulse (NaN too)
      const double gf = u * fma(u, fma(u, p.g3, p.g2), p.g1);
      const int gfx = __double2loint(__dadd_rd(gf, kMagicFx));   // floor(gf * 2^20)
      const int g0 = gfx >> kFracBits;
      if (g0 < -1 || g0 >= G) continue;                           // the window margin of the pre-test
      const float w1 = (float)(gfx & (kFxOne - 1)) * p.w_scale;
      const float fr = cycles_fraction(fma(gf, p.cq, p.fr0));
      const float gfxf = (float)gfx;
      const float inv_R2 = fmaf(gfxf, fmaf(gfxf, p.a2, p.a1), p.a0);
      const float p1 = fmaf(s_p1v[i], tf, s_p1[i]), p2 = fmaf(s_p2v[i], tf, s_p2[i]);
      const float A = amp * ex2_approx(fmaf(p2, p2, p1 * p1) * (inv_R2 * p.neg_alpha_log2e)) * inv_R2;
      float sn, cs;
      __sincosf(6.283185307179586f * fr, &sn, &cs);
      const float re = A * cs, im = -A * sn;
      if (__float_as_int(A) <= hi_bits) {   // native int32 adds (a warp's lanes hit different rows: no same-address replay)
        const float w1s = w1 * sc, w0s = sc - w1s;
        const unsigned a0 = row_a + 8u * (unsigned)g0;
        if (g0 >= 0) {
          asm volatile("red.shared.add.s32 [%0], %1;" ::"r"(a0), "r"(__float_as_int(fmaf(re, w0s, 12582912.0f)) - 0x4B400000) : "memory");
          asm volatile("red.shared.add.s32 [%0+4], %1;" ::"r"(a0), "r"(__float_as_int(fmaf(im, w0s, 12582912.0f)) - 0x4B400000) : "memory");
        }
        if (g0 + 1 < G) {
          asm volatile("red.shared.add.s32 [%0+8], %1;" ::"r"(a0), "r"(__float_as_int(fmaf(re, w1s, 12582912.0f)) - 0x4B400000) : "memory");
          asm volatile("red.shared.add.s32 [%0+12], %1;" ::"r"(a0), "r"(__float_as_int(fmaf(im, w1s, 12582912.0f)) - 0x4B400000) : "memory");
        }
      } else {   // brighter than the fixed-point range admits: exact fp32 reduction in global memory (rare)
        const float w0 = 1.0f - w1;
        float2* y = rp.Y + ((size_t)blockIdx.x * kRegJT + lane) * G;
        if (g0 >= 0) atomicAdd(&y[g0], make_float2(w0 * re, w0 * im));
        if (g0 + 1 < G) atomicAdd(&y[g0 + 1], make_float2(w1 * re, w1 * im));
      }
    }
  }
  flush();
}

cudaError_t launch_regular(const AccParams& a, float2* Y, long long j0, int n_pulses, double prf, int sm_count,
                           size_t smem_optin, cudaStream_t st, int* launches) {
  if (n_pulses <= 0 || a.n == 0) return cudaSuccess;
  const size_t smem = regular_smem_bytes(a.G);
  if (smem > smem_optin - 2048) return cudaErrorInvalidConfiguration;
  cudaError_t e = cudaFuncSetAttribute(regular_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return e;
  RegParams rp;
  rp.a = a;
  rp.Y = Y;
  rp.j0 = j0;
  rp.n_pulses = n_pulses;
  rp.prf = prf;
  const int tiles = (n_pulses + kRegJT - 1) / kRegJT;
  int slices = (4 * sm_count + tiles - 1) / tiles;   // about four blocks per SM in total
  const unsigned long long max_slices = (a.n + kRegChunk - 1) / kRegChunk;
  if ((unsigned long long)slices > max_slices) slices = (int)max_slices;
  if (slices > 65535) slices = 65535;
  if (slices < 1) slices = 1;
  rp.n_slices = slices;
  regular_kernel<<<dim3(tiles, slices), kRegThreads, smem, st>>>(rp);
  ++*launches;
  return cudaGetLastError();
}

}  // namespace simk
