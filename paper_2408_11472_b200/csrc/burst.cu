// Delay-Doppler burst step (reading R8): the IQ stream is split
// into bursts of B pulses and every burst gets an along-track FFT per range gate:
//     Z[b][k][g] = sum_{m<B} Y[b B + m][g] exp(-2 pi i k m / B),   unnormalised, k in natural order.
// A second batched-FFT workload next to the synthesis kernel, with the transform along the SLOW axis of Y.
// One block = one burst x a tile of 32 gates: the B x 32 samples are read gate-fastest (coalesced), stored
// transposed in shared memory ([gate][pulse], row padded), transformed in place by the same decimation-in-frequency
// radix-4 passes as synthesize.cu with conjugated twiddles, and written back gate-fastest from the bit-reversed rows.
#include "sim_internal.h"

namespace simk {

constexpr int kBurstThreads = 256;
constexpr int kBurstGates = 32;   // gates per block

__device__ __forceinline__ float2 bmul(float2 a, float2 b) {
  return make_float2(fmaf(a.x, b.x, -a.y * b.y), fmaf(a.x, b.y, a.y * b.x));
}
__device__ __forceinline__ float2 badd(float2 a, float2 b) { return make_float2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ float2 bsub(float2 a, float2 b) { return make_float2(a.x - b.x, a.y - b.y); }
__device__ __forceinline__ float2 bmulni(float2 a) { return make_float2(a.y, -a.x); }   // -i * a

template <int LOGB>
__global__ void __launch_bounds__(kBurstThreads) burst_fft_kernel(const float2* __restrict__ Y, float2* __restrict__ Z,
                                                                   int G) {
  constexpr int B = 1 << LOGB, LD = B + 1;
  __shared__ float2 tw[B / 2];                  // exp(-2 pi i j / B)
  __shared__ float2 sig[kBurstGates * LD];      // [gate][pulse]
  const int tid = threadIdx.x;
  const long long burst = blockIdx.x;
  const int gbase = blockIdx.y * kBurstGates;
  const int rows = min(kBurstGates, G - gbase);
  for (int j = tid; j < B / 2; j += kBurstThreads) {
    float s, c;
    sincospif(-2.0f * (float)j / (float)B, &s, &c);   // exact arguments: j / B is dyadic
    tw[j] = make_float2(c, s);
  }
  const float2* src = Y + (size_t)burst * B * G + gbase;
  for (int e = tid; e < B * kBurstGates; e += kBurstThreads) {
    const int m = e >> 5, g = e & 31;
    if (g < rows) sig[g * LD + m] = src[(size_t)m * G + g];
  }
  __syncthreads();

  int q = LOGB;
#pragma unroll 1
  for (; q >= 2; q -= 2) {   // stages of distance 2h and h fused (h = 2^(q-2)), forward transform
    const int h = 1 << (q - 2);
    const int shq = LOGB - q, shh = LOGB - q + 1;
    for (int e = tid; e < kBurstGates * (B / 4); e += kBurstThreads) {
      const int g = e >> (LOGB - 2), t = e & (B / 4 - 1);
      if (g >= rows) continue;
      const int j = t & (h - 1);
      float2* x = sig + g * LD + (((t >> (q - 2)) << q) + j);
      const float2 wq = tw[j << shq], wh = tw[j << shh];
      const float2 x0 = x[0], x1 = x[h], x2 = x[2 * h], x3 = x[3 * h];
      const float2 a0 = badd(x0, x2), a2 = bmul(bsub(x0, x2), wq);
      const float2 a1 = badd(x1, x3), a3 = bmulni(bmul(bsub(x1, x3), wq));   // twiddle W^(j+h) = -i W^j (forward)
      x[0] = badd(a0, a1);
      x[h] = bmul(bsub(a0, a1), wh);
      x[2 * h] = badd(a2, a3);
      x[3 * h] = bmul(bsub(a2, a3), wh);
    }
    __syncthreads();
  }
  if (q == 1) {
    for (int e = tid; e < kBurstGates * (B / 2); e += kBurstThreads) {
      const int g = e >> (LOGB - 1), t = e & (B / 2 - 1);
      if (g >= rows) continue;
      float2* x = sig + g * LD + 2 * t;
      const float2 a = x[0], b = x[1];
      x[0] = badd(a, b);
      x[1] = bsub(a, b);
    }
    __syncthreads();
  }

  float2* dst = Z + (size_t)burst * B * G + gbase;
  for (int e = tid; e < B * kBurstGates; e += kBurstThreads) {
    const int k = e >> 5, g = e & 31;
    if (g < rows) dst[(size_t)k * G + g] = sig[g * LD + (int)(__brev((unsigned)k) >> (32 - LOGB))];
  }
}

cudaError_t launch_burst_fft(const float2* Y, float2* Z, long long n_bursts, int logB, int G, cudaStream_t st,
                             int* launches) {
  if (n_bursts <= 0) return cudaSuccess;
  const int gy = (G + kBurstGates - 1) / kBurstGates;
  long long done = 0;
  while (done < n_bursts) {
    const int nx = (int)((n_bursts - done) < 0x7fffffffLL ? (n_bursts - done) : 0x7fffffffLL);
    const dim3 grid(nx, gy);
    const float2* y = Y + (size_t)done * ((size_t)1 << logB) * G;
    float2* z = Z + (size_t)done * ((size_t)1 << logB) * G;
    switch (logB) {
      case 4: burst_fft_kernel<4><<<grid, kBurstThreads, 0, st>>>(y, z, G); break;
      case 5: burst_fft_kernel<5><<<grid, kBurstThreads, 0, st>>>(y, z, G); break;
      case 6: burst_fft_kernel<6><<<grid, kBurstThreads, 0, st>>>(y, z, G); break;
      case 7: burst_fft_kernel<7><<<grid, kBurstThreads, 0, st>>>(y, z, G); break;
      default: return cudaErrorInvalidValue;
    }
    ++*launches;
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    done += nx;
  }
  return cudaSuccess;
}

}  // namespace simk
