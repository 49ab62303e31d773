// Steps S1-S3: post-processing of the fast mode in one kernel.
//   S1  batched inverse DFT along Doppler of the spectra: hand-written shared-memory Stockham
//       (autosort) FFT with radix-4, -2, -3 and -5 passes, so any N = 2^a 3^b 5^c runs exactly (the paper's update
//       intervals n_fast = 250 ... 1250, as N = P or N = 2P); unnormalised, kernel exp(+2 pi i k m / N);
//   S2  weighting with eq. (1) and sum of the two long-time signals;
//   S3  write of the IQ block Y[x][g], pulse-major, gate fastest.
// One block = a tile of GT gates x a run of consecutive segments: the long-time signal y_{s+1} of a segment is kept in
// shared memory and serves as y_s of the next one, so every spectrum is transformed once per run (not twice), and the
// IQ rows are written in pieces of GT gates (64 bytes for GT = 8).
#include "sim_internal.h"

namespace simk {

constexpr int kSynThreads = 256;

// tw[j] = exp(+2 pi i j / N), j < N
__global__ void twiddle_kernel(float2* tw, int N) {
  const int j = blockIdx.x * blockDim.x + threadIdx.x;
  if (j < N) {
    double s, c;
    sincospi(2.0 * (double)j / (double)N, &s, &c);
    tw[j] = make_float2((float)c, (float)s);
  }
}

cudaError_t launch_twiddles(float2* tw, int N, cudaStream_t st, int* launches) {
  twiddle_kernel<<<(N + 127) / 128, 128, 0, st>>>(tw, N);
  ++*launches;
  return cudaGetLastError();
}

// N = 2^a 3^b 5^c -> passes (radix 4 first, then one 2, then 3s and 5s); false when N has another prime factor
bool synth_factor(int N, int* radix, int* n_pass) {
  int n = N, k = 0;
  while (n % 4 == 0) { radix[k++] = 4; n /= 4; }
  while (n % 2 == 0) { radix[k++] = 2; n /= 2; }
  while (n % 3 == 0) { radix[k++] = 3; n /= 3; }
  while (n % 5 == 0) { radix[k++] = 5; n /= 5; }
  *n_pass = k;
  return n == 1 && k <= kSynMaxPass;
}

constexpr int kSynMaxWeightTable = 4096;   // pulses per update up to which eq. (1) is tabulated once per block
static int synth_weight_entries(int P) { return P <= kSynMaxWeightTable ? P : 0; }
size_t synth_smem_bytes(int N, int GT, int P) { return ((size_t)3 * GT * (N + 1) + N + synth_weight_entries(P)) * sizeof(float2); }

// Gates per block and segments per block.  Three signal buffers of GT rows must fit; a long call (many segments)
// uses 8-gate tiles (64-byte IQ pieces) and runs of segments that still give about two blocks per SM; a short call
// takes smaller tiles so that it has blocks at all.
void synth_plan(int N, int G, int P, long long n_segments, int sm_count, int* gt_out, int* seg_per_block) {
  int gt = 8;
  while (gt > 1 && synth_smem_bytes(N, gt, P) > 100 * 1024) gt >>= 1;
  while (gt > 2 && n_segments * ((G + gt - 1) / gt) < sm_count / 2) gt >>= 1;
  const long long tiles = (G + gt - 1) / gt;
  long long runs = (2LL * sm_count + tiles - 1) / tiles;   // runs of segments wanted per gate tile
  if (runs < 1) runs = 1;
  if (runs > n_segments) runs = n_segments;
  *gt_out = gt;
  *seg_per_block = (int)((n_segments + runs - 1) / runs);
}

__device__ __forceinline__ float2 cmul(float2 a, float2 b) {
  return make_float2(fmaf(a.x, b.x, -a.y * b.y), fmaf(a.x, b.y, a.y * b.x));
}
__device__ __forceinline__ float2 cadd(float2 a, float2 b) { return make_float2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ float2 csub(float2 a, float2 b) { return make_float2(a.x - b.x, a.y - b.y); }
__device__ __forceinline__ float2 cmuli(float2 a) { return make_float2(-a.y, a.x); }   // i * a
__device__ __forceinline__ float2 cscale(float2 a, float s) { return make_float2(a.x * s, a.y * s); }

// R-point inverse DFT (kernel exp(+2 pi i a b / R)) in place
template <int R>
__device__ __forceinline__ void idft_small(float2* v);
template <>
__device__ __forceinline__ void idft_small<2>(float2* v) {
  const float2 a = v[0], b = v[1];
  v[0] = cadd(a, b);
  v[1] = csub(a, b);
}
template <>
__device__ __forceinline__ void idft_small<4>(float2* v) {
  const float2 a0 = cadd(v[0], v[2]), a1 = csub(v[0], v[2]), b0 = cadd(v[1], v[3]), b1 = cmuli(csub(v[1], v[3]));
  v[0] = cadd(a0, b0);
  v[1] = cadd(a1, b1);
  v[2] = csub(a0, b0);
  v[3] = csub(a1, b1);
}
template <>
__device__ __forceinline__ void idft_small<3>(float2* v) {
  const float s3 = 0.8660254037844386f;   // sin(2 pi / 3)
  const float2 t = cadd(v[1], v[2]), d = cscale(cmuli(csub(v[1], v[2])), s3);
  const float2 m = make_float2(v[0].x - 0.5f * t.x, v[0].y - 0.5f * t.y);
  v[0] = cadd(v[0], t);
  v[1] = cadd(m, d);
  v[2] = csub(m, d);
}
template <>
__device__ __forceinline__ void idft_small<5>(float2* v) {
  const float c1 = 0.30901699437494745f, c2 = -0.8090169943749475f;   // cos(2 pi / 5), cos(4 pi / 5)
  const float s1 = 0.9510565162951535f, s2 = 0.5877852522924731f;     // sin(2 pi / 5), sin(4 pi / 5)
  const float2 t1 = cadd(v[1], v[4]), t2 = cadd(v[2], v[3]), d1 = csub(v[1], v[4]), d2 = csub(v[2], v[3]);
  const float2 m1 = make_float2(v[0].x + c1 * t1.x + c2 * t2.x, v[0].y + c1 * t1.y + c2 * t2.y);
  const float2 m2 = make_float2(v[0].x + c2 * t1.x + c1 * t2.x, v[0].y + c2 * t1.y + c1 * t2.y);
  const float2 e1 = cmuli(make_float2(s1 * d1.x + s2 * d2.x, s1 * d1.y + s2 * d2.y));
  const float2 e2 = cmuli(make_float2(s2 * d1.x - s1 * d2.x, s2 * d1.y - s1 * d2.y));
  v[0] = cadd(v[0], cadd(t1, t2));
  v[1] = cadd(m1, e1);
  v[4] = csub(m1, e1);
  v[2] = cadd(m2, e2);
  v[3] = csub(m2, e2);
}

// One Stockham pass of radix R over `rows` signals of N points: src -> dst (rows LD apart).  Ns = product of the
// radices already done.  Butterfly j < N/R reads src[j + t N/R], twiddles by W_{Ns R}^{(j mod Ns) t}, writes
// dst[(j - j mod Ns) R + (j mod Ns) + t Ns].  POW2: N/R and Ns are powers of two (every index is a shift or a mask).
template <int R, bool POW2>
__device__ __forceinline__ void stockham_pass(const float2* __restrict__ src, float2* __restrict__ dst, const float2* __restrict__ tw,
                                              int rows, int M, int LD, int Ns, int tstep, int tid) {
  // M = N / R butterflies per signal; tstep = M / Ns: twiddle index k t N / (Ns R) < N needs no reduction
  const int logM = 31 - __clz(M);
  for (int e = tid; e < rows * M; e += kSynThreads) {
    const int row = POW2 ? (e >> logM) : (e / M), j = POW2 ? (e & (M - 1)) : (e - row * M);
    const int k = POW2 ? (j & (Ns - 1)) : (j % Ns);
    const float2* s = src + (size_t)row * LD + j;
    float2 v[R];
#pragma unroll
    for (int t = 0; t < R; ++t) v[t] = s[t * M];
    if (Ns > 1) {
#pragma unroll
      for (int t = 1; t < R; ++t) v[t] = cmul(v[t], tw[k * t * tstep]);
    }
    idft_small<R>(v);
    float2* d = dst + (size_t)row * LD + (j - k) * R + k;
#pragma unroll
    for (int t = 0; t < R; ++t) d[t * Ns] = v[t];
  }
}

__global__ void __launch_bounds__(kSynThreads) synth_kernel(SynParams p) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int N = p.N, LD = N + 1, GT = p.GT;
  float2* tw = reinterpret_cast<float2*>(smem_raw);   // [N] exp(+2 pi i j / N)
  float2* buf0 = tw + N;                              // three signal buffers [GT][N+1]
  const size_t bufsz = (size_t)GT * LD;
  const int tid = threadIdx.x;
  const int gbase = blockIdx.y * GT;
  const int rows = min(GT, p.G - gbase);
  const long long s_begin = p.seg0 + (long long)blockIdx.x * p.seg_per_block;
  const long long s_end = min(s_begin + p.seg_per_block, p.seg0 + p.n_segments);

  for (int j = tid; j < N; j += kSynThreads) tw[j] = p.tw[j];
  // eq. (1) for every pulse offset of a segment, once per block: wt[m] = (W_s, W_{s+1}) at a = m / P
  const int P = p.P;
  const float invP = 1.0f / (float)P;
  float2* wt = buf0 + 3 * bufsz;
  const bool tabulated = P <= kSynMaxWeightTable;
  auto weights = [&](int m) {
    const float a = (float)m * invP;
    float ws = 1.0f - a, wn = a;
    if (p.weight_mode == SIM_W_SQRT) {
      ws = sqrtf(ws);
      wn = sqrtf(wn);
    }
    return make_float2(ws, wn);
  };
  if (tabulated)
    for (int m = tid; m < P; m += kSynThreads) wt[m] = weights(m);

  const bool pow2 = (N & (N - 1)) == 0;
  const int logGT = 31 - __clz(GT), logN = 31 - __clz(N);
  // S1 of spectrum u: rows of T_u -> buffer `a` (straight copy), passes between `a` and `b`; returns where y_u ended up
  auto transform = [&](long long u, float2* a, float2* b) -> float2* {
    const float2* T = p.ring + (size_t)(u % p.cap) * p.slot_stride + (size_t)gbase * N;
    // batches of eight loads per thread in flight before the first store (the rows of a tile are contiguous in T)
    const int total = rows * N;
    for (int base = tid; base < total; base += 8 * kSynThreads) {
      float2 r[8];
#pragma unroll
      for (int i = 0; i < 8; ++i) {
        const int e = base + i * kSynThreads;
        if (e < total) r[i] = __ldg(T + e);
      }
#pragma unroll
      for (int i = 0; i < 8; ++i) {
        const int e = base + i * kSynThreads;
        if (e < total) {
          const int rw = pow2 ? (e >> logN) : (e / N);
          a[(size_t)rw * LD + (e - rw * N)] = r[i];
        }
      }
    }
    __syncthreads();
    for (int ps = 0; ps < p.n_pass; ++ps) {
      const int R = p.radix[ps], M = p.pass_m[ps], Ns = p.pass_ns[ps], ts = p.pass_tstep[ps];
      if (pow2) {
        if (R == 4) stockham_pass<4, true>(a, b, tw, rows, M, LD, Ns, ts, tid);
        else stockham_pass<2, true>(a, b, tw, rows, M, LD, Ns, ts, tid);
      } else {
        if (R == 4) stockham_pass<4, false>(a, b, tw, rows, M, LD, Ns, ts, tid);
        else if (R == 2) stockham_pass<2, false>(a, b, tw, rows, M, LD, Ns, ts, tid);
        else if (R == 3) stockham_pass<3, false>(a, b, tw, rows, M, LD, Ns, ts, tid);
        else stockham_pass<5, false>(a, b, tw, rows, M, LD, Ns, ts, tid);
      }
      __syncthreads();
      float2* t = a; a = b; b = t;
    }
    return a;
  };

  float2* cur = buf0;
  float2* f1 = buf0 + bufsz;
  float2* f2 = buf0 + 2 * bufsz;
  {
    float2* r = transform(s_begin, cur, f1);
    if (r != cur) { f1 = cur; cur = r; }
  }
  // one thread = one gate row of the tile and every (256 / GT)-th pulse of the segment: row, base pointers and the
  // output stride are loop invariants, the sample indices advance by additions
  const int row = tid & (GT - 1), pi0 = tid >> logGT, pstep = kSynThreads >> logGT;
  const size_t ostep = (size_t)pstep * p.G;
  int off_n = (-P) % N;            // (m - P) mod N = (m + off_n) mod N, off_n in [0, N)
  off_n += off_n < 0 ? N : 0;
  const int pstep_n = pstep % N;
  for (long long s = s_begin; s < s_end; ++s) {
    const bool has_next = (s + 1 < p.n_spectra);
    float2* nxt = nullptr;
    if (has_next) {
      nxt = transform(s + 1, f1, f2);
      if (nxt != f1) { f2 = f1; f1 = nxt; }   // (f1 now names the buffer holding y_{s+1}; f2 the free one)
    }
    // ---- S2 + S3: cross-fade and write, gate fastest ----
    const long long seg_lo = s * (long long)P;
    const long long lo = max(seg_lo, p.x0), hi = min(seg_lo + P, p.x0 + p.n_pulses);
    const int npul = (int)(hi - lo);
    if (row < rows) {
      const float2* crow = cur + (size_t)row * LD;
      const float2* nrow = has_next ? nxt + (size_t)row * LD : crow;
      float2* outp = p.iq + (size_t)(lo - p.x0 + pi0) * p.G + gbase + row;
      int m = (int)(lo - seg_lo) + pi0;   // 0..P-1
      int ms = m % N;
      for (int pi = pi0; pi < npul; pi += pstep, m += pstep, outp += ostep) {
        const float2 ys = crow[ms];
        float2 out = ys;   // tail rule: a lone spectrum at weight 1
        if (has_next) {
          int mn = ms + off_n;
          mn -= mn >= N ? N : 0;
          const float2 yn = nrow[mn];
          const float2 w = tabulated ? wt[m] : weights(m);
          out = make_float2(w.x * ys.x + w.y * yn.x, w.x * ys.y + w.y * yn.y);
        }
        *outp = out;
        ms += pstep_n;
        ms -= ms >= N ? N : 0;
      }
    }
    __syncthreads();   // the emission has read `cur`: it becomes a free buffer
    if (has_next) {
      float2* t = cur; cur = f1; f1 = t;
    }
  }
}

// Once per handle: the dynamic shared-memory limit of the kernel (largest plan for this N).
cudaError_t synth_prepare(int N, int P) {
  int gt = 8;
  while (gt > 1 && synth_smem_bytes(N, gt, P) > 100 * 1024) gt >>= 1;
  return cudaFuncSetAttribute(synth_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)synth_smem_bytes(N, gt, P));
}

cudaError_t launch_synthesize(const SynParams& p0, cudaStream_t st, int* launches) {
  if (p0.n_segments <= 0 || p0.n_pulses <= 0) return cudaSuccess;
  SynParams p = p0;
  if (!synth_factor(p.N, p.radix, &p.n_pass)) return cudaErrorInvalidValue;
  for (int ps = 0, ns = 1; ps < p.n_pass; ns *= p.radix[ps], ++ps) {   // per-pass constants of the Stockham scheme
    p.pass_m[ps] = p.N / p.radix[ps];
    p.pass_ns[ps] = ns;
    p.pass_tstep[ps] = p.pass_m[ps] / ns;
  }
  const size_t smem = synth_smem_bytes(p.N, p.GT, p.P);
  // per launch: the limit is per function and per device, another handle may have set it for a smaller N
  cudaError_t e = cudaFuncSetAttribute(synth_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return e;
  const int gy = (p.G + p.GT - 1) / p.GT;
  const long long runs = (p.n_segments + p.seg_per_block - 1) / p.seg_per_block;
  long long done = 0;
  while (done < runs) {   // gridDim.x can be large for long tracks
    const long long nx = (runs - done) < (1LL << 30) ? (runs - done) : (1LL << 30);
    SynParams q = p;
    q.seg0 = p.seg0 + done * p.seg_per_block;
    q.n_segments = p.n_segments - done * p.seg_per_block;
    if (q.n_segments > nx * p.seg_per_block) q.n_segments = nx * p.seg_per_block;
    synth_kernel<<<dim3((unsigned)nx, gy), kSynThreads, smem, st>>>(q);
    ++*launches;
    e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    done += nx;
  }
  return cudaSuccess;
}

}  // namespace simk
