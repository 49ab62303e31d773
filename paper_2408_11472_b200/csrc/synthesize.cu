// Steps S1-S3: post-processing of the fast mode in one kernel.
//   S1  batched inverse DFT along Doppler of the spectra of updates s and s+1,
//       hand-written shared-memory FFT (decimation in frequency; radix-4 passes = two fused radix-2 stages,
//       one radix-2 pass when log2 N is odd; natural-order load, bit-reversed read in the epilogue),
//       unnormalised, kernel exp(+2 pi i k m / N);
//   S2  weighting with eq. (1) and sum of the two long-time signals;
//   S3  write of the IQ block Y[x][g], pulse-major, gate fastest.
// One block = one segment s (pulses sP .. (s+1)P-1) x one tile of GT gates (GT a power of two).  N is a
// template parameter: every index is a shift or a mask.
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

int synth_gate_tile(int N, int G, long long n_segments, int sm_count) {
  // two signals x GT rows x (N+1) float2 (+ the twiddle table) must fit comfortably in shared memory ...
  int gt = 16;
  while (gt > 1 && (size_t)2 * gt * (N + 1) * sizeof(float2) > 160 * 1024) gt >>= 1;
  // ... and the grid should give every SM several blocks: a call is a few segments x G gates, so small gate tiles
  // are what gives it blocks.  Not below 2 gates (16-byte pieces of the gate-fastest IQ rows).
  while (gt > 2 && n_segments * ((G + gt - 1) / gt) < 8LL * sm_count) gt >>= 1;
  return gt;
}

__device__ __forceinline__ float2 cmul(float2 a, float2 b) {
  return make_float2(fmaf(a.x, b.x, -a.y * b.y), fmaf(a.x, b.y, a.y * b.x));
}
__device__ __forceinline__ float2 cadd(float2 a, float2 b) { return make_float2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ float2 csub(float2 a, float2 b) { return make_float2(a.x - b.x, a.y - b.y); }
__device__ __forceinline__ float2 cmuli(float2 a) { return make_float2(-a.y, a.x); }   // i * a

template <int LOGN>
__global__ void __launch_bounds__(kSynThreads) synth_kernel(SynParams p) {
  constexpr int N = 1 << LOGN, LD = N + 1, HALF_N = N / 2;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  float2* tw = reinterpret_cast<float2*>(smem_raw);   // [N/2] exp(+2 pi i j / N)
  float2* sig = tw + HALF_N;                          // [2][GT][N+1]
  const int GT = p.GT, logGT = 31 - __clz(GT);
  const long long s = p.seg0 + blockIdx.x;
  const int gbase = blockIdx.y * GT;
  const int rows = min(GT, p.G - gbase);
  const bool has_next = (s + 1 < p.n_spectra);
  const int nsig = has_next ? 2 : 1;
  const int tid = threadIdx.x;

  // ---- twiddles and spectra rows into shared memory, natural order: a straight, conflict-free copy ----
  for (int j = tid; j < HALF_N; j += kSynThreads) tw[j] = p.tw[j];
  for (int w = 0; w < nsig; ++w) {
    const float2* T = p.ring + (size_t)((s + w) % p.cap) * p.slot_stride + (size_t)gbase * N;
    float2* dst = sig + (size_t)w * GT * LD;
    for (int e = tid; e < rows * N; e += kSynThreads) dst[(e >> LOGN) * LD + (e & (N - 1))] = T[e];
  }
  __syncthreads();

  // ---- S1: decimation in frequency, in place over all nsig * GT signals (rows beyond `rows` are skipped);
  //      natural-order input, BIT-REVERSED output: y[m] ends up at index brev(m) ----
  const int nsignals = nsig << logGT;
  int q = LOGN;   // the next pass works inside blocks of 2^q elements
#pragma unroll 1
  for (; q >= 2; q -= 2) {   // stages of distance 2h and h fused (h = 2^(q-2)): elements i0 + {0, h, 2h, 3h}
    const int h = 1 << (q - 2);
    const int shq = LOGN - q, shh = LOGN - q + 1;   // twiddle index steps N / 4h and N / 2h
    for (int e = tid; e < nsignals * (N / 4); e += kSynThreads) {
      const int sidx = e >> (LOGN - 2), t = e & (N / 4 - 1);
      if ((sidx & (GT - 1)) >= rows) continue;
      const int j = t & (h - 1);
      float2* x = sig + (size_t)sidx * LD + (((t >> (q - 2)) << q) + j);
      const float2 wq = tw[j << shq], wh = tw[j << shh];
      const float2 x0 = x[0], x1 = x[h], x2 = x[2 * h], x3 = x[3 * h];
      const float2 a0 = cadd(x0, x2), a2 = cmul(csub(x0, x2), wq);
      const float2 a1 = cadd(x1, x3), a3 = cmuli(cmul(csub(x1, x3), wq));   // twiddle W_4h^(j+h) = i W_4h^j
      x[0] = cadd(a0, a1);
      x[h] = cmul(csub(a0, a1), wh);
      x[2 * h] = cadd(a2, a3);
      x[3 * h] = cmul(csub(a2, a3), wh);
    }
    __syncthreads();
  }
  if (q == 1) {  // log2 N odd: the last stage (distance 1, twiddle 1) on its own
    for (int e = tid; e < nsignals * HALF_N; e += kSynThreads) {
      const int sidx = e >> (LOGN - 1), t = e & (HALF_N - 1);
      if ((sidx & (GT - 1)) >= rows) continue;
      float2* x = sig + (size_t)sidx * LD + 2 * t;
      const float2 a = x[0], b = x[1];
      x[0] = cadd(a, b);
      x[1] = csub(a, b);
    }
    __syncthreads();
  }

  // ---- S2 + S3: cross-fade and write, gate fastest ----
  const long long seg_lo = s * (long long)p.P;
  const long long lo = max(seg_lo, p.x0), hi = min(seg_lo + p.P, p.x0 + p.n_pulses);
  const int npul = (int)(hi - lo);
  const float invP = 1.0f / (float)p.P;
  for (int e = tid; e < (npul << logGT); e += kSynThreads) {
    const int pi = e >> logGT, row = e & (GT - 1);
    if (row >= rows) continue;
    const long long x = lo + pi;
    const int m = (int)(x - seg_lo);  // 0..P-1
    const float2 ys = sig[(size_t)row * LD + (int)(__brev((unsigned)(m & (N - 1))) >> (32 - LOGN))];
    float2 out;
    if (has_next) {
      const float a = (float)m * invP;
      float ws = 1.0f - a, wn = a;
      if (p.weight_mode == SIM_W_SQRT) {
        ws = sqrtf(ws);
        wn = sqrtf(wn);
      }
      const float2 yn = sig[((size_t)GT + row) * LD + (int)(__brev((unsigned)((m - p.P) & (N - 1))) >> (32 - LOGN))];
      out = make_float2(ws * ys.x + wn * yn.x, ws * ys.y + wn * yn.y);
    } else {
      out = ys;  // tail rule: lone spectrum at weight 1
    }
    p.iq[(size_t)(x - p.x0) * p.G + gbase + row] = out;
  }
}

typedef void (*SynKernel)(SynParams);

static SynKernel syn_kernel(int logN) {
  switch (logN) {
    case 4: return synth_kernel<4>;
    case 5: return synth_kernel<5>;
    case 6: return synth_kernel<6>;
    case 7: return synth_kernel<7>;
    case 8: return synth_kernel<8>;
    case 9: return synth_kernel<9>;
    case 10: return synth_kernel<10>;
    case 11: return synth_kernel<11>;
    default: return nullptr;
  }
}

size_t synth_smem_bytes(int N, int GT) { return ((size_t)2 * GT * (N + 1) + N / 2) * sizeof(float2); }

// Once per handle: the dynamic shared-memory limit of the kernel for this N (largest gate tile).
cudaError_t synth_prepare(int logN) {
  SynKernel k = syn_kernel(logN);
  if (!k) return cudaErrorInvalidValue;
  const int N = 1 << logN;
  return cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize,
                              (int)synth_smem_bytes(N, synth_gate_tile(N, 1, 1 << 30, 1)));
}

cudaError_t launch_synthesize(const SynParams& p, int n_segments, cudaStream_t st, int* launches) {
  if (n_segments <= 0 || p.n_pulses <= 0) return cudaSuccess;
  SynKernel k = syn_kernel(p.logN);
  if (!k) return cudaErrorInvalidValue;
  const size_t smem = synth_smem_bytes(p.N, p.GT);
  // gridDim.x (segments) can be large for long tracks; gridDim.y (gate tiles) <= 1024
  const int gy = (p.G + p.GT - 1) / p.GT;
  int done = 0;
  while (done < n_segments) {
    const int nx = (n_segments - done) < 65535 * 32 ? (n_segments - done) : 65535 * 32;
    SynParams q = p;
    q.seg0 = p.seg0 + done;
    k<<<dim3(nx, gy), kSynThreads, smem, st>>>(q);
    ++*launches;
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    done += nx;
  }
  return cudaSuccess;
}

}  // namespace simk
