// Steps S1-S3: post-processing of the fast mode in one kernel.
//   S1  batched inverse DFT along Doppler of the spectra of updates s and s+1,
//       hand-written shared-memory radix-2 FFT, unnormalised, kernel exp(+2 pi i k m / N);
//   S2  weighting with eq. (1) and sum of the two long-time signals;
//   S3  write of the IQ block Y[x][g], pulse-major, gate fastest.
// One block = one segment s (pulses sP .. (s+1)P-1) x one tile of GT gates.
#include "sim_internal.h"

namespace simk {

constexpr int kSynThreads = 256;

__global__ void twiddle_kernel(float2* tw, int N) {
  const int j = blockIdx.x * blockDim.x + threadIdx.x;
  if (j < N / 2) {
    double s, c;
    sincospi(2.0 * (double)j / (double)N, &s, &c);
    tw[j] = make_float2((float)c, (float)s);
  }
}

cudaError_t launch_twiddles(float2* tw, int N, cudaStream_t st, int* launches) {
  twiddle_kernel<<<(N / 2 + 127) / 128, 128, 0, st>>>(tw, N);
  ++*launches;
  return cudaGetLastError();
}

int synth_gate_tile(int N) {
  // two signals x GT rows x (N+1) float2 must fit comfortably in shared memory
  int gt = 16;
  while (gt > 1 && (size_t)2 * gt * (N + 1) * sizeof(float2) > 160 * 1024) gt >>= 1;
  return gt;
}

__device__ __forceinline__ float2 cmul(float2 a, float2 b) {
  return make_float2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
}

__global__ void __launch_bounds__(kSynThreads) synth_kernel(SynParams p) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  float2* sig = reinterpret_cast<float2*>(smem_raw);  // [2][GT][N+1]
  const int N = p.N, GT = p.GT, ld = N + 1;
  const long long s = p.seg0 + blockIdx.x;
  const int gbase = blockIdx.y * GT;
  const int rows = min(GT, p.G - gbase);
  const bool has_next = (s + 1 < p.n_spectra);
  const int nsig = has_next ? 2 : 1;
  const int tid = threadIdx.x;

  // ---- load spectra rows into shared memory in bit-reversed order (coalesced along Doppler) ----
  for (int w = 0; w < nsig; ++w) {
    const float2* T = p.ring + (size_t)((s + w) % p.cap) * p.slot_stride + (size_t)gbase * N;
    float2* dst = sig + (size_t)w * GT * ld;
    for (int e = tid; e < rows * N; e += kSynThreads) {
      const int row = e / N, k = e - row * N;
      const int kr = (int)(__brev((unsigned)k) >> (32 - p.logN));
      dst[row * ld + kr] = T[(size_t)row * N + k];
    }
  }
  __syncthreads();

  // ---- S1: in-place radix-2 decimation-in-time stages over all nsig*rows signals ----
  const int half_total = nsig * rows * (N / 2);
  for (int st = 1; st <= p.logN; ++st) {
    const int half = 1 << (st - 1);
    const int tw_step = (N / 2) >> (st - 1);
    for (int e = tid; e < half_total; e += kSynThreads) {
      const int sidx = e / (N / 2);          // which signal (w * rows + row)
      const int t = e - sidx * (N / 2);
      const int w = sidx / rows, row = sidx - w * rows;
      float2* xsig = sig + ((size_t)w * GT + row) * ld;
      const int j = t & (half - 1);
      const int i0 = ((t >> (st - 1)) << st) + j;
      const int i1 = i0 + half;
      const float2 a = xsig[i0];
      const float2 b = cmul(xsig[i1], p.tw[j * tw_step]);
      xsig[i0] = make_float2(a.x + b.x, a.y + b.y);
      xsig[i1] = make_float2(a.x - b.x, a.y - b.y);
    }
    __syncthreads();
  }

  // ---- S2 + S3: cross-fade and write, gate fastest ----
  const long long seg_lo = s * (long long)p.P;
  const long long lo = max(seg_lo, p.x0), hi = min(seg_lo + p.P, p.x0 + p.n_pulses);
  const int npul = (int)(hi - lo);
  const float invP = 1.0f / (float)p.P;
  for (int e = tid; e < npul * rows; e += kSynThreads) {
    const int pi = e / rows, row = e - pi * rows;
    const long long x = lo + pi;
    const int m = (int)(x - seg_lo);  // 0..P-1
    const float2 ys = sig[(size_t)row * ld + (m & (N - 1))];
    float2 out;
    if (has_next) {
      const float a = (float)m * invP;
      float ws = 1.0f - a, wn = a;
      if (p.weight_mode == SIM_W_SQRT) {
        ws = sqrtf(ws);
        wn = sqrtf(wn);
      }
      const float2 yn = sig[((size_t)GT + row) * ld + ((m - p.P) & (N - 1))];
      out = make_float2(ws * ys.x + wn * yn.x, ws * ys.y + wn * yn.y);
    } else {
      out = ys;  // tail rule: lone spectrum at weight 1
    }
    p.iq[(size_t)(x - p.x0) * p.G + gbase + row] = out;
  }
}

cudaError_t launch_synthesize(const SynParams& p, int n_segments, cudaStream_t st, int* launches) {
  if (n_segments <= 0 || p.n_pulses <= 0) return cudaSuccess;
  const size_t smem = (size_t)2 * p.GT * (p.N + 1) * sizeof(float2);
  cudaError_t e = cudaFuncSetAttribute(synth_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return e;
  // gridDim.x (segments) can be large for long tracks; gridDim.y (gate tiles) <= 1024
  const int gy = (p.G + p.GT - 1) / p.GT;
  int done = 0;
  while (done < n_segments) {
    const int nx = (n_segments - done) < 65535 * 32 ? (n_segments - done) : 65535 * 32;
    SynParams q = p;
    q.seg0 = p.seg0 + done;
    synth_kernel<<<dim3(nx, gy), kSynThreads, smem, st>>>(q);
    ++*launches;
    e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    done += nx;
  }
  return cudaSuccess;
}

}  // namespace simk
