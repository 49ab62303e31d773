// REGULAR MODE (reading R5): the surface is updated at every
// pulse and the raw data of a pulse are the complex sum of all scatterers per range gate.  Scatterers and
// satellite in uniform motion from the states given at pulse 0:
//     Y[j][g] = sum_p w_g(R_p(t_j)) sqrt(s0dA_p) G(theta_p(t_j)) / R_p(t_j)^2 exp(-i 4 pi R_p(t_j) / lambda),  t_j = j / PRF.
// Work = scatterers x pulses.  No Doppler axis, no FFT: this is the at-scale truth the fast mode approximates.
//
// One THREAD = one PULSE with a private row Y[j][0..G) in shared memory (plain read-modify-write, no atomics);
// a block = JT pulses x one slice of the scatterers.  The block's threads first turn a chunk of scatterers into
// per-scatterer constants (u(t) = R(t)^2 - rg0^2 = u0 + a t + b t^2 in fp64, antenna projections linear in t),
// then every thread walks the chunk (shared-memory broadcasts).  Per (scatterer, pulse): 2 DFMA for u, the gate
// coordinate by the same polynomial as the fast-mode index path, phase fraction in fp64, the rest in fp32.
// At the end the block adds its tile to Y with red.global.add.v2.f32.
#include "scatter_math.cuh"

namespace simk {

constexpr int kRegChunk = 256;   // scatterers per shared-memory chunk

struct RegParams {
  AccParams a;       // geometry constants (make_acc_params)
  float2* Y;         // [n_pulses][G]
  long long j0;      // first pulse, relative to the instant of the satellite state
  int n_pulses, JT;  // pulses of the call, pulses (= threads) per block
  int n_slices;      // scatterer slices (gridDim.y)
  double prf;        // t_j = j / PRF, the oracle's expression
};

size_t regular_smem_bytes(int G, int JT) {
  return (size_t)JT * (2 * G + 1) * sizeof(float) + (size_t)kRegChunk * (3 * sizeof(double) + 6 * sizeof(float));
}

__global__ void regular_kernel(RegParams rp) {
  const AccParams& p = rp.a;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int G = p.G, JT = rp.JT, LD = 2 * G + 1;
  double* s_u0 = reinterpret_cast<double*>(smem_raw);   // [chunk] u at pulse 0
  double* s_a = s_u0 + kRegChunk;                        // [chunk] 2 d.dv
  double* s_b = s_a + kRegChunk;                         // [chunk] |dv|^2
  float* s_p1 = reinterpret_cast<float*>(s_b + kRegChunk);   // [chunk] d.e1, then dv.e1, d.e2, dv.e2, sqrt(s0dA), live
  float* s_p1v = s_p1 + kRegChunk;
  float* s_p2 = s_p1v + kRegChunk;
  float* s_p2v = s_p2 + kRegChunk;
  float* s_amp = s_p2v + kRegChunk;
  float* s_pad = s_amp + kRegChunk;                      // (unused sixth array keeps the tile 8-byte aligned)
  float* tile = s_pad + kRegChunk;                       // [JT][2G+1]: re, im interleaved per gate
  const int tid = threadIdx.x;
  float* row = tile + (size_t)tid * LD;
  for (int i = 0; i < LD; ++i) row[i] = 0.0f;

  const long long j = rp.j0 + (long long)blockIdx.x * JT + tid;
  const bool pulse_ok = (long long)blockIdx.x * JT + tid < rp.n_pulses;
  const double t = __ddiv_rn((double)j, rp.prf);
  const float tf = (float)t;

  const unsigned long long per = (p.n + rp.n_slices - 1) / rp.n_slices;
  const unsigned long long lo = per * blockIdx.y, hi = (lo + per < p.n) ? lo + per : p.n;
  // Each thread prepares up to kPrep scatterers of a chunk.  Their raw inputs are fetched into registers one chunk
  // ahead, so that the global-load latency is hidden behind the evaluation of the current chunk.
  constexpr int kPrep = (kRegChunk + 31) / 32;   // enough for the smallest block (32 threads)
  float in[kPrep][7];
  auto fetch = [&](unsigned long long base) {
#pragma unroll
    for (int k = 0; k < kPrep; ++k) {
      const unsigned long long q = base + tid + (unsigned long long)k * JT;
      const bool v = tid + k * JT < kRegChunk && q < hi;
      in[k][0] = v ? p.x[q] : 0.0f; in[k][1] = v ? p.y[q] : 0.0f; in[k][2] = v ? p.z[q] : 0.0f;
      in[k][3] = v ? p.vx[q] : 0.0f; in[k][4] = v ? p.vy[q] : 0.0f; in[k][5] = v ? p.vz[q] : 0.0f;
      in[k][6] = v ? p.s0dA[q] : 0.0f;
    }
  };
  if (lo < hi) fetch(lo);
  for (unsigned long long base = lo; base < hi; base += kRegChunk) {
    const int m = (int)((hi - base < (unsigned long long)kRegChunk) ? hi - base : kRegChunk);
    __syncthreads();   // the previous chunk has been consumed
#pragma unroll
    for (int k = 0; k < kPrep; ++k) {
      const int i = tid + k * JT;
      if (i >= m) continue;
      const float s0 = in[k][6];
      const double dx = __dsub_rn((double)in[k][0], p.sx), dy = __dsub_rn((double)in[k][1], p.sy), dz = __dsub_rn((double)in[k][2], p.sz);
      const double dvx = (double)in[k][3] - p.svx, dvy = (double)in[k][4] - p.svy, dvz = (double)in[k][5] - p.svz;
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
    if (base + kRegChunk < hi) fetch(base + kRegChunk);   // in flight during the evaluation below
    if (!pulse_ok) continue;
#pragma unroll 2
    for (int i = 0; i < m; ++i) {
      const float amp = s_amp[i];
      const double u = fma(t, fma(t, s_b[i], s_a[i]), s_u0[i]);
      if (!(amp > 0.0f) || !(u >= p.uw_lo && u <= p.uw_hi)) continue;   // dead, or outside the window (NaN too)
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
      const float re = A * cs, im = -A * sn, w0 = 1.0f - w1;
      if (g0 >= 0) {
        row[2 * g0] = fmaf(w0, re, row[2 * g0]);
        row[2 * g0 + 1] = fmaf(w0, im, row[2 * g0 + 1]);
      }
      if (g0 + 1 < G) {
        row[2 * g0 + 2] = fmaf(w1, re, row[2 * g0 + 2]);
        row[2 * g0 + 3] = fmaf(w1, im, row[2 * g0 + 3]);
      }
    }
  }
  __syncthreads();
  // ---- flush: gate fastest across threads so that the reductions of a warp hit consecutive addresses ----
  const int rows = min(JT, rp.n_pulses - blockIdx.x * JT);
  for (int e = tid; e < rows * G; e += JT) {
    const int r = e / G, g = e - r * G;
    const float re = tile[(size_t)r * LD + 2 * g], im = tile[(size_t)r * LD + 2 * g + 1];
    if (re != 0.0f || im != 0.0f) atomicAdd(&rp.Y[((size_t)blockIdx.x * JT + r) * G + g], make_float2(re, im));
  }
}

cudaError_t launch_regular(const AccParams& a, float2* Y, long long j0, int n_pulses, double prf, int sm_count,
                           size_t smem_optin, cudaStream_t st, int* launches) {
  if (n_pulses <= 0 || a.n == 0) return cudaSuccess;
  int JT = 192;
  while (JT > 32 && (JT - 32 >= n_pulses || regular_smem_bytes(a.G, JT) > smem_optin - 2048)) JT -= 32;
  if (regular_smem_bytes(a.G, JT) > smem_optin - 2048) return cudaErrorInvalidConfiguration;
  const size_t smem = regular_smem_bytes(a.G, JT);
  cudaError_t e = cudaFuncSetAttribute(regular_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return e;
  RegParams rp;
  rp.a = a;
  rp.Y = Y;
  rp.j0 = j0;
  rp.n_pulses = n_pulses;
  rp.JT = JT;
  rp.prf = prf;
  const int tiles = (n_pulses + JT - 1) / JT;
  int slices = (2 * sm_count + tiles - 1) / tiles;
  const unsigned long long max_slices = (a.n + kRegChunk - 1) / kRegChunk;
  if ((unsigned long long)slices > max_slices) slices = (int)max_slices;
  if (slices > 65535) slices = 65535;
  rp.n_slices = slices;
  regular_kernel<<<dim3(tiles, slices), JT, smem, st>>>(rp);
  ++*launches;
  return cudaGetLastError();
}

}  // namespace simk
