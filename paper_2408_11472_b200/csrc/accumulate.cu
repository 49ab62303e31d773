// Steps A1-A7: scatterer -> (gate, Doppler bin, complex amplitude) -> spectrum T_u[G][N].
// Paper: Algorithm 1 body and `rasterize`.  sm_100a, no tensor cores: the step is a
// streaming scan (28 B per scatterer) with a scatter-add, bounded by HBM, the fp64 pipe and the
// shared-memory atomic unit.  Design notes and measurements: DESIGN.md "Kernels".
#include <climits>

#include "sim_internal.h"

namespace simk {

// 1.5 * 2^(52 - kFracBits): adding it to v (|v| < 2^11) leaves floor/round(v * 2^20) in the low word.
constexpr double kMagicFx = 6442450944.0;        // 1.5 * 2^32
constexpr double kMagicFxHalf = 6442450944.5;    // the same + 0.5 (nearest-bin rule, ties up)
constexpr double kMagicPhase = 402653184.0;      // 1.5 * 2^28: low word = round(q * 2^24)
constexpr int kFxOne = 1 << kFracBits;
constexpr float kFxScale = 1.0f / (float)kFxOne;

struct Geo {
  int g0, k;     // gate of the lower half in [-1, G-1], Doppler bin in [0, N)
  float w1;      // weight of gate g0+1 (gate g0 gets 1 - w1)
  float fr;      // frac(2R/lambda) mapped to [-0.5, 0.5) cycles
  float delta;   // R - rg0, metres
};

__device__ __forceinline__ float phase_fraction(double two_over_lambda, double fr0, double delta) {
  // 2R/lambda = 2 rg0/lambda + 2 delta/lambda; only the fraction matters (phase = -2 pi frac)
  const double q = __fma_rn(delta, two_over_lambda, fr0);
  const int lo = __double2loint(__dadd_rn(q, kMagicPhase));
  return (float)(int)((unsigned)lo << 8) * 2.3283064365386963e-10f;  // * 2^-32
}

// ---------------------------------------------------------------------------------------------
// CANONICAL fp64 INDEX SEQUENCE of DESIGN.md, continued from dx, dy, dz, R2 (which every path
// computes identically).  Explicit round-to-nearest intrinsics: nvcc must not contract a*b+c
// differently from the definition.  Kept out of line (the fast path calls it only inside the guard
// band) and fed by value, so that the kernel parameters stay in constant memory.
// Returns (g0, k, bits of w1, bits of fr); g0 = SIM_GATE_NONE when the scatterer is dropped.
// ---------------------------------------------------------------------------------------------
struct CanonConsts {
  double rg0, inv_dR, cD, two_over_lambda, fr0, svx, svy, svz;
  int G, N;
};

__device__ __noinline__ int4 canonical_tail(CanonConsts c, double dx, double dy, double dz, double R2,
                                            float vxf, float vyf, float vzf) {
  const int4 dropped = make_int4(SIM_GATE_NONE, -1, 0, 0);
  const double R = __dsqrt_rn(R2);
  const double delta = __dsub_rn(R, c.rg0);
  const double gf = __dmul_rn(delta, c.inv_dR);
  if (!(gf >= -1.0 && gf < (double)c.G)) return dropped;  // touches no gate (NaN lands here too)
  const double g0d = floor(gf);
  const double dvx = __dsub_rn((double)vxf, c.svx);
  const double dvy = __dsub_rn((double)vyf, c.svy);
  const double dvz = __dsub_rn((double)vzf, c.svz);
  const double rdot = __ddiv_rn(__fma_rn(dvz, dz, __fma_rn(dvy, dy, __dmul_rn(dvx, dx))), R);
  const double kf = __dmul_rn(rdot, c.cD);
  if (!(fabs(kf) < 1073741824.0)) return dropped;
  const double kk = floor(__dadd_rn(kf, 0.5));
  // N is a power of two: two's-complement AND is the mathematical mod
  return make_int4((int)g0d, ((int)kk) & (c.N - 1), __float_as_int((float)__dsub_rn(gf, g0d)),
                   __float_as_int(phase_fraction(c.two_over_lambda, c.fr0, delta)));
}

__device__ __forceinline__ bool canonical(const AccParams& p, double dx, double dy, double dz, double R2,
                                          float vxf, float vyf, float vzf, Geo& o) {
  CanonConsts c;
  c.rg0 = p.rg0; c.inv_dR = p.inv_dR; c.cD = p.cD; c.two_over_lambda = p.two_over_lambda; c.fr0 = p.fr0;
  c.svx = p.svx; c.svy = p.svy; c.svz = p.svz; c.G = p.G; c.N = p.N;
  const int4 r = canonical_tail(c, dx, dy, dz, R2, vxf, vyf, vzf);
  if (r.x == SIM_GATE_NONE) return false;
  o.g0 = r.x;
  o.k = r.y;
  o.w1 = __int_as_float(r.z);
  o.fr = __int_as_float(r.w);
  o.delta = ((float)r.x + o.w1) * p.dR_f;
  return true;
}

// Steps A2-A4.  index_path 0: canonical sequence for every scatterer.  index_path 1: delta = R - rg0 from
// u = R^2 - rg0^2 by a 4-term series and 1/R by a 3-term series (no sqrt, no divide), gate and bin from
// 2^-20 fixed point; whenever a coordinate lies within `guard` of a boundary the canonical sequence decides.
__device__ __forceinline__ bool geometry(const AccParams& p, float xf, float yf, float zf, float vxf,
                                         float vyf, float vzf, Geo& o, unsigned& fallbacks) {
  const double dx = __dsub_rn((double)xf, p.sx);
  const double dy = __dsub_rn((double)yf, p.sy);
  const double dz = __dsub_rn((double)zf, p.sz);
  const double R2 = __fma_rn(dz, dz, __fma_rn(dy, dy, __dmul_rn(dx, dx)));
  if (!(p.index_path && p.fast_ok)) return canonical(p, dx, dy, dz, R2, vxf, vyf, vzf, o);

  const double u = (R2 - p.rg0sq_hi) - p.rg0sq_lo;
  if (!(u >= p.u_lo && u <= p.u_hi)) return false;  // certainly outside the window (or NaN)
  const double t = u * p.inv_2rg0;
  const double delta = t * fma(t, fma(t, fma(t, p.b3, p.b2), p.b1), 1.0);
  const int gfx = __double2loint(__dadd_rd(delta * p.inv_dR, kMagicFx));   // floor(gf * 2^20)
  const int gfrac = gfx & (kFxOne - 1);
  const double dvx = (double)vxf - p.svx, dvy = (double)vyf - p.svy, dvz = (double)vzf - p.svz;
  const double num = __fma_rn(dvz, dz, __fma_rn(dvy, dy, __dmul_rn(dvx, dx)));
  const double e = delta * p.inv_rg0;
  const double inv_R = p.inv_rg0 * fma(-e, fma(-e, 1.0 - e, 1.0), 1.0);   // 1/(rg0 (1+e)) to e^4
  const double kf = (num * inv_R) * p.cD;
  const int kfx = __double2loint(__dadd_rd(kf, kMagicFxHalf));             // floor((kf + 0.5) * 2^20)
  const int kfrac = kfx & (kFxOne - 1);
  const unsigned span = (unsigned)(kFxOne - 2 * p.guard);
  const bool near = (unsigned)(gfrac - p.guard) >= span || (unsigned)(kfrac - p.guard) >= span ||
                    !(fabs(kf) < 1024.0);
  if (near) {
    ++fallbacks;
    return canonical(p, dx, dy, dz, R2, vxf, vyf, vzf, o);
  }
  const int g0 = gfx >> kFracBits;
  if (g0 < -1 || g0 >= p.G) return false;
  o.g0 = g0;
  o.k = (kfx >> kFracBits) & (p.N - 1);
  o.w1 = (float)gfrac * kFxScale;
  o.fr = phase_fraction(p.two_over_lambda, p.fr0, delta);
  o.delta = (float)gfx * p.dR_fx;
  return true;
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

// Step A5: sqrt(s0dA) G(theta) / R^2 exp(-i 2 pi fr), all fp32.  Returns |c| too.
__device__ __forceinline__ float2 amplitude(const AccParams& p, const Geo& g, float xf, float yf, float zf,
                                            float s0dA, float& A) {
  const float dx = (xf - p.sxh) - p.sxl, dy = (yf - p.syh) - p.syl, dz = (zf - p.szh) - p.szl;
  const float e = g.delta * p.inv_rg0_f;
  const float inv_R2 = p.inv_rg0sq_f * fmaf(e, fmaf(e, 3.0f, -2.0f), 1.0f);  // 1/(rg0 (1+e))^2 to e^3
  const float cx = dy * p.bz - dz * p.by;
  const float cy = dz * p.bx - dx * p.bz;
  const float cz = dx * p.by - dy * p.bx;
  const float sin2 = (cx * cx + cy * cy + cz * cz) * inv_R2;
  A = sqrt_approx(s0dA) * ex2_approx(p.neg_alpha_log2e * sin2) * inv_R2;
  float sn, cs;
  __sincosf(6.283185307179586f * g.fr, &sn, &cs);
  return make_float2(A * cs, -A * sn);
}

// ---------------------------------------------------------------------------------------------
// Variant 0: reference kernel.  One scatterer per thread, global fp32x2 reductions into T.
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) acc_reference_kernel(AccParams p) {
  const unsigned long long stride = (unsigned long long)gridDim.x * blockDim.x;
  unsigned fb = 0;
  for (unsigned long long i = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; i < p.n;
       i += stride) {
    const float s0 = p.s0dA[i];
    if (!(s0 > 0.0f)) continue;
    Geo g;
    const float xf = p.x[i], yf = p.y[i], zf = p.z[i];
    if (!geometry(p, xf, yf, zf, p.vx[i], p.vy[i], p.vz[i], g, fb)) continue;
    float A;
    const float2 c = amplitude(p, g, xf, yf, zf, s0, A);
    const float w1 = g.w1, w0 = 1.0f - w1;
    if (g.g0 >= 0) atomicAdd(&p.T[(size_t)g.g0 * p.N + g.k], make_float2(w0 * c.x, w0 * c.y));
    if (g.g0 + 1 < p.G) atomicAdd(&p.T[(size_t)(g.g0 + 1) * p.N + g.k], make_float2(w1 * c.x, w1 * c.y));
  }
}

// ---------------------------------------------------------------------------------------------
// Index-only kernel (parity pin P11): runs the same index routine as the production kernel.
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) indices_kernel(AccParams p, int32_t* __restrict__ g0,
                                                      int32_t* __restrict__ k) {
  const unsigned long long stride = (unsigned long long)gridDim.x * blockDim.x;
  unsigned fb = 0;
  for (unsigned long long i = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; i < p.n;
       i += stride) {
    Geo g;
    if (geometry(p, p.x[i], p.y[i], p.z[i], p.vx[i], p.vy[i], p.vz[i], g, fb)) {
      g0[i] = g.g0;
      k[i] = g.k;
    } else {
      g0[i] = SIM_GATE_NONE;
      k[i] = -1;
    }
  }
  if (fb) atomicAdd(&p.counters[kCtrFallback], fb);
}

// ---------------------------------------------------------------------------------------------
// Variant 1: shared-memory tile kernel (the production path).
//
//  * Persistent blocks draw "super-chunks" of consecutive scatterers from a ticket counter and stream
//    them in chunks of 1024 (4 per thread, 128-bit loads, next chunk prefetched in registers).
//  * sm_100a has no native shared-memory fp32 atomic add (it is an LDS + ATOMS.CAST.SPIN loop that
//    collapses under the contention of this workload: 10^3..10^4 scatterers per populated cell), but
//    ATOMS.ADD on int32 is native.  Each chunk is therefore one block-floating-point EPOCH:
//      phase 1  geometry + amplitude of the thread's 4 scatterers, kept in registers; block statistics
//               (count, mean amplitude, Doppler-offset range, gate range) by REDUX/shuffles + 5 ATOMS;
//      phase 2  contributions scaled by s = 2^e with mean*s in [2^16, 2^17) and added with ATOMS.ADD to an
//               int32 tile [G][W]; a component above 2^20 or a bin outside the window "escapes" to a
//               global fp32x2 reduction (exact, rare).  <= 1024 adds of <= 2^20 per cell: no overflow.
//      drain    touched rows of the int tile -> fp32 tile (x 2^-e), int tile zeroed.
//    Quantisation: LSB = 2^-e <= mean * 2^-16, so the relative L2 error of an epoch is <= 0.82 * 2^-16
//    = 1.3e-5 whatever the amplitude distribution (mean <= rms); see DESIGN.md.
//  * The Doppler window [k0, k0+W) follows the data: the chunk's own bin range (known after phase 1)
//    decides whether the window holds or moves (fp32 tile flushed to T with global reductions, step A7).
// ---------------------------------------------------------------------------------------------
struct ChunkStats {
  int dmin, dmax;   // signed circular Doppler offset from the window centre
  int gmin, gmax;   // g0 range
  int anyk;         // the bin of some scatterer of the chunk
  int cnt;          // illuminated scatterers
  float wsum[kAccWarps];  // per-warp sum of |c|
};

__device__ __forceinline__ void stats_reset(ChunkStats& s) {
  s.dmin = INT_MAX;
  s.dmax = INT_MIN;
  s.gmin = INT_MAX;
  s.gmax = INT_MIN;
  s.anyk = 0;
  s.cnt = 0;
}

struct Contrib {
  int code;  // -1: nothing; else (g0 + 1) | (k << 11)
  float w1, re, im;
};

struct Quad {
  float4 x, y, z, vx, vy, vz, s;
};

__device__ __forceinline__ float4 ldg_stream(const float* ptr) {
  float4 v;
  asm volatile("ld.global.nc.L1::no_allocate.v4.f32 {%0,%1,%2,%3}, [%4];"
               : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w)
               : "l"(ptr));
  return v;
}

__device__ __forceinline__ void load_quad(const AccParams& p, unsigned long long i, Quad& q) {
  q.x = ldg_stream(p.x + i);
  q.y = ldg_stream(p.y + i);
  q.z = ldg_stream(p.z + i);
  q.vx = ldg_stream(p.vx + i);
  q.vy = ldg_stream(p.vy + i);
  q.vz = ldg_stream(p.vz + i);
  q.s = ldg_stream(p.s0dA + i);
}

__device__ __forceinline__ float4 ldg_ragged(const float* a, unsigned long long i, unsigned long long end) {
  float4 v;
  v.x = (i + 0 < end) ? a[i + 0] : 0.0f;
  v.y = (i + 1 < end) ? a[i + 1] : 0.0f;
  v.z = (i + 2 < end) ? a[i + 2] : 0.0f;
  v.w = (i + 3 < end) ? a[i + 3] : 0.0f;
  return v;
}

// last, partial group of four of the input: missing entries read as s0dA = 0 (contribute nothing)
__device__ __forceinline__ void load_ragged(const AccParams& p, unsigned long long i, unsigned long long end,
                                            Quad& q) {
  q.x = ldg_ragged(p.x, i, end);
  q.y = ldg_ragged(p.y, i, end);
  q.z = ldg_ragged(p.z, i, end);
  q.vx = ldg_ragged(p.vx, i, end);
  q.vy = ldg_ragged(p.vy, i, end);
  q.vz = ldg_ragged(p.vz, i, end);
  q.s = ldg_ragged(p.s0dA, i, end);
}

__device__ __forceinline__ void phase1_one(const AccParams& p, float xf, float yf, float zf, float vxf,
                                           float vyf, float vzf, float s0, Contrib& c, float& A,
                                           unsigned& fallbacks) {
  c.code = -1;
  A = 0.0f;
  if (!(s0 > 0.0f)) return;
  Geo g;
  if (!geometry(p, xf, yf, zf, vxf, vyf, vzf, g, fallbacks)) return;
  const float2 v = amplitude(p, g, xf, yf, zf, s0, A);
  c.code = (g.g0 + 1) | (g.k << 11);
  c.w1 = g.w1;
  c.re = v.x;
  c.im = v.y;
}

__device__ __forceinline__ void tile_flush(const AccParams& p, float2* tile_f, int k0, int logW) {
  const int cells = p.G << logW;
  for (int c = threadIdx.x; c < cells; c += kAccThreads) {
    const float2 f = tile_f[c];
    if (f.x != 0.0f || f.y != 0.0f) {
      tile_f[c] = make_float2(0.0f, 0.0f);
      const int g = c >> logW, kw = c & (p.W - 1);
      atomicAdd(&p.T[(size_t)g * p.N + ((k0 + kw) & (p.N - 1))], f);
    }
  }
}

__global__ void __launch_bounds__(kAccThreads, 2) acc_tile_kernel(AccParams p) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int cells = p.G * p.W;
  int2* tile_i = reinterpret_cast<int2*>(smem_raw);
  float2* tile_f = reinterpret_cast<float2*>(smem_raw + (size_t)cells * sizeof(int2));
  __shared__ ChunkStats s_stats[3];
  __shared__ unsigned long long s_ticket;

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int N = p.N, W = p.W, halfW = W >> 1;
  const int logW = 31 - __clz(W);
  for (int c = tid; c < cells; c += kAccThreads) {
    tile_i[c] = make_int2(0, 0);
    tile_f[c] = make_float2(0.0f, 0.0f);
  }
  if (tid < 3) stats_reset(s_stats[tid]);

  const unsigned long long n_sc = (p.n + p.superchunk - 1) / p.superchunk;
  int kc = (W >= N) ? (N >> 1) : 0;   // window centre; the window is [kc - W/2, kc + W/2) mod N
  bool tile_has_data = false;
  unsigned escapes = 0, flushes = 0, fallbacks = 0;
  unsigned chunk_no = 0;              // selects the rotating statistics set

  for (;;) {
    __syncthreads();  // previous super-chunk (incl. its last drain) finished; s_ticket free
    if (tid == 0) s_ticket = atomicAdd(&p.counters[kCtrTicket], 1u);
    __syncthreads();
    const unsigned long long sc = s_ticket;
    if (sc >= n_sc) break;
    const unsigned long long base = sc * p.superchunk;
    const unsigned long long end = (base + p.superchunk < p.n) ? base + p.superchunk : p.n;

    unsigned long long i = base + (unsigned long long)tid * kAccPerThread;
    Quad cur;
    if (i + kAccPerThread <= end) load_quad(p, i, cur);
    else load_ragged(p, i, end, cur);

    for (unsigned long long cb = base; cb < end; cb += kAccChunk, ++chunk_no) {
      // ---- prefetch the next chunk ----
      const unsigned long long inext = i + kAccChunk;
      Quad nxt;
      if (cb + kAccChunk < end) {
        if (inext + kAccPerThread <= end) load_quad(p, inext, nxt);
        else load_ragged(p, inext, end, nxt);
      }

      // ---- phase 1: geometry + amplitude, block statistics ----
      Contrib c[4];
      float A[4];
      phase1_one(p, cur.x.x, cur.y.x, cur.z.x, cur.vx.x, cur.vy.x, cur.vz.x, cur.s.x, c[0], A[0], fallbacks);
      phase1_one(p, cur.x.y, cur.y.y, cur.z.y, cur.vx.y, cur.vy.y, cur.vz.y, cur.s.y, c[1], A[1], fallbacks);
      phase1_one(p, cur.x.z, cur.y.z, cur.z.z, cur.vx.z, cur.vy.z, cur.vz.z, cur.s.z, c[2], A[2], fallbacks);
      phase1_one(p, cur.x.w, cur.y.w, cur.z.w, cur.vx.w, cur.vy.w, cur.vz.w, cur.s.w, c[3], A[3], fallbacks);

      ChunkStats& st = s_stats[chunk_no % 3u];
      int cnt = 0, dmin = INT_MAX, dmax = INT_MIN, gmin = INT_MAX, gmax = INT_MIN, anyk = 0;
      float sumA = 0.0f;
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        if (c[j].code >= 0) {
          const int k = c[j].code >> 11, g0 = (c[j].code & 2047) - 1;
          const int d = ((k - kc + (N >> 1)) & (N - 1)) - (N >> 1);
          dmin = min(dmin, d);
          dmax = max(dmax, d);
          gmin = min(gmin, g0);
          gmax = max(gmax, g0);
          anyk = k;
          ++cnt;
          sumA += A[j];
        }
      }
      const unsigned live = __ballot_sync(0xffffffffu, cnt > 0);
      if (live) {  // warp-uniform
        dmin = __reduce_min_sync(0xffffffffu, dmin);
        dmax = __reduce_max_sync(0xffffffffu, dmax);
        gmin = __reduce_min_sync(0xffffffffu, gmin);
        gmax = __reduce_max_sync(0xffffffffu, gmax);
        cnt = __reduce_add_sync(0xffffffffu, cnt);
        anyk = __shfl_sync(0xffffffffu, anyk, __ffs(live) - 1);
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) sumA += __shfl_xor_sync(0xffffffffu, sumA, o);
        if (lane == 0) {
          atomicMin(&st.dmin, dmin);
          atomicMax(&st.dmax, dmax);
          atomicMin(&st.gmin, gmin);
          atomicMax(&st.gmax, gmax);
          atomicAdd(&st.cnt, cnt);
          st.anyk = anyk;
        }
      }
      if (lane == 0) st.wsum[warp] = live ? sumA : 0.0f;
      __syncthreads();  // (A) statistics complete; every drain of the previous chunk has finished
      if (tid == 0) stats_reset(s_stats[(chunk_no + 2u) % 3u]);  // last read one chunk ago, next written after the next (A)

      const int tot = st.cnt;
      if (tot > 0) {  // block-uniform
        // ---- place the Doppler window ----
        const int bdmin = st.dmin, bdmax = st.dmax;
        if (!(bdmin >= -halfW && bdmax <= halfW - 1)) {
          const int kc_new = ((bdmax - bdmin < W) ? kc + ((bdmin + bdmax) >> 1) : st.anyk) & (N - 1);
          if (tile_has_data) {
            tile_flush(p, tile_f, (kc - halfW) & (N - 1), logW);  // int tile is empty here
            ++flushes;
            tile_has_data = false;
          }
          kc = kc_new;
        }
        const int k0 = (kc - halfW) & (N - 1);

        // ---- block-floating-point scale of this epoch: mean * s in [2^16, 2^17) ----
        float tsum = 0.0f;
#pragma unroll
        for (int w = 0; w < kAccWarps; ++w) tsum += st.wsum[w];
        const float mean = tsum / (float)tot;
        int ex = 16 - (((__float_as_int(mean) >> 23) & 0xff) - 127);
        ex = max(-126, min(127, ex));
        const float s = __int_as_float((ex + 127) << 23);
        const float inv_s = __int_as_float((127 - ex) << 23);
        const float lim = 1048575.0f / s;  // |component| * s <= 2^20 - 1

        // ---- phase 2: native int32 shared-memory atomics ----
#pragma unroll
        for (int j = 0; j < 4; ++j) {
          if (c[j].code < 0) continue;
          const int k = c[j].code >> 11, g0 = (c[j].code & 2047) - 1;
          const unsigned kw = (unsigned)(k - k0) & (unsigned)(N - 1);
          const float w1 = c[j].w1, w0 = 1.0f - w1;
          const float2 v0 = make_float2(w0 * c[j].re, w0 * c[j].im);
          const float2 v1 = make_float2(w1 * c[j].re, w1 * c[j].im);
          if (kw < (unsigned)W && fmaxf(fabsf(c[j].re), fabsf(c[j].im)) <= lim) {
            if (g0 >= 0) {
              int2* cell = &tile_i[(g0 << logW) + (int)kw];
              atomicAdd(&cell->x, __float2int_rn(v0.x * s));
              atomicAdd(&cell->y, __float2int_rn(v0.y * s));
            }
            if (g0 + 1 < p.G) {
              int2* cell = &tile_i[((g0 + 1) << logW) + (int)kw];
              atomicAdd(&cell->x, __float2int_rn(v1.x * s));
              atomicAdd(&cell->y, __float2int_rn(v1.y * s));
            }
          } else {
            if (g0 >= 0) atomicAdd(&p.T[(size_t)g0 * N + k], v0);
            if (g0 + 1 < p.G) atomicAdd(&p.T[(size_t)(g0 + 1) * N + k], v1);
            ++escapes;
          }
        }
        __syncthreads();  // (B) all atomics of the epoch landed

        // ---- drain: touched rows of the int tile -> fp32 tile ----
        const int r0 = max(st.gmin, 0), r1 = min(st.gmax + 1, p.G - 1);
        const int dbase = r0 << logW, dcells = (r1 - r0 + 1) << logW;
        for (int cc = tid; cc < dcells; cc += kAccThreads) {
          const int2 v = tile_i[dbase + cc];
          if (v.x | v.y) {
            tile_i[dbase + cc] = make_int2(0, 0);
            float2 f = tile_f[dbase + cc];
            f.x = fmaf((float)v.x, inv_s, f.x);
            f.y = fmaf((float)v.y, inv_s, f.y);
            tile_f[dbase + cc] = f;
          }
        }
        tile_has_data = true;
      }
      cur = nxt;
      i = inext;
    }
  }

  // the loop is left right after a barrier that follows every drain
  if (tile_has_data) {
    tile_flush(p, tile_f, (kc - halfW) & (N - 1), logW);
    ++flushes;
  }
  if (escapes) atomicAdd(&p.counters[kCtrEscape], escapes);
  if (fallbacks) atomicAdd(&p.counters[kCtrFallback], fallbacks);
  if (tid == 0 && flushes) atomicAdd(&p.counters[kCtrFlush], flushes);
}

// ---------------------------------------------------------------------------------------------
// Launchers
// ---------------------------------------------------------------------------------------------
size_t acc_tile_smem_bytes(int G, int W) { return (size_t)G * W * (sizeof(int2) + sizeof(float2)); }

cudaError_t acc_tile_blocks_per_sm(int G, int W, int* blocks) {
  const size_t smem = acc_tile_smem_bytes(G, W);
  cudaError_t e = cudaFuncSetAttribute(acc_tile_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return e;
  return cudaOccupancyMaxActiveBlocksPerMultiprocessor(blocks, acc_tile_kernel, kAccThreads, smem);
}

cudaError_t launch_accumulate(const AccParams& p, int variant, int blocks, cudaStream_t st,
                              int* launches) {
  if (p.n == 0) return cudaSuccess;
  if (variant == 0) {
    unsigned long long want = (p.n + 255) / 256;
    const unsigned long long cap = (unsigned long long)blocks * 8;
    const int grid = (int)(want < cap ? want : cap);
    acc_reference_kernel<<<grid, 256, 0, st>>>(p);
    ++*launches;
    return cudaGetLastError();
  }
  const size_t smem = acc_tile_smem_bytes(p.G, p.W);
  cudaError_t e = cudaFuncSetAttribute(acc_tile_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return e;
  e = cudaMemsetAsync(p.counters + kCtrTicket, 0, sizeof(unsigned int), st);
  if (e != cudaSuccess) return e;
  const unsigned long long n_sc = (p.n + p.superchunk - 1) / p.superchunk;
  const int grid = (int)(n_sc < (unsigned long long)blocks ? n_sc : (unsigned long long)blocks);
  acc_tile_kernel<<<grid, kAccThreads, smem, st>>>(p);
  ++*launches;
  return cudaGetLastError();
}

cudaError_t launch_indices(const AccParams& p, int32_t* g0, int32_t* k, cudaStream_t st, int* launches) {
  if (p.n == 0) return cudaSuccess;
  unsigned long long want = (p.n + 255) / 256;
  const int grid = (int)(want < 148ull * 16 ? want : 148ull * 16);
  indices_kernel<<<grid, 256, 0, st>>>(p, g0, k);
  ++*launches;
  return cudaGetLastError();
}

}  // namespace simk
