// Steps A1-A7: scatterer -> (gate, Doppler bin, complex amplitude) -> spectrum T_u[G][N].
// Paper: Algorithm 1 body and `rasterize`.  sm_100a, no tensor cores: the step is a
// streaming scan (28 B per scatterer) with a scatter-add, bounded by HBM and by the fp64 pipe.
#include "sim_internal.h"

namespace simk {

// ---------------------------------------------------------------------------------------------
// Geometry of one scatterer.  The index part is the CANONICAL fp64 SEQUENCE of DESIGN.md: explicit
// round-to-nearest intrinsics so that nvcc cannot contract a*b+c differently from the definition.
// ---------------------------------------------------------------------------------------------
struct Geo {
  int g0, k;
  float w1;          // weight of gate g0+1 (gate g0 gets 1 - w1)
  double R2, fr;     // squared range; frac(2R/lambda) in [0,1)
  double dx, dy, dz;
};

__device__ __forceinline__ bool canonical_geometry(const AccParams& p, float xf, float yf, float zf,
                                                   float vxf, float vyf, float vzf, Geo& o) {
  const double dx = __dsub_rn((double)xf, p.sx);
  const double dy = __dsub_rn((double)yf, p.sy);
  const double dz = __dsub_rn((double)zf, p.sz);
  const double R2 = __fma_rn(dz, dz, __fma_rn(dy, dy, __dmul_rn(dx, dx)));
  const double R = __dsqrt_rn(R2);
  const double gf = __dmul_rn(__dsub_rn(R, p.rg0), p.inv_dR);
  if (!(gf >= -1.0 && gf < (double)p.G)) return false;  // touches no gate (NaN lands here too)
  const double g0d = floor(gf);
  const double dvx = __dsub_rn((double)vxf, p.svx);
  const double dvy = __dsub_rn((double)vyf, p.svy);
  const double dvz = __dsub_rn((double)vzf, p.svz);
  const double rdot = __ddiv_rn(__fma_rn(dvz, dz, __fma_rn(dvy, dy, __dmul_rn(dvx, dx))), R);
  const double kf = __dmul_rn(rdot, p.cD);
  if (!(fabs(kf) < 1073741824.0)) return false;
  const double kk = floor(__dadd_rn(kf, 0.5));
  const double q = __dmul_rn(R, p.two_over_lambda);
  o.g0 = (int)g0d;
  o.k = ((int)kk) & (p.N - 1);  // N is a power of two: two's-complement AND is the mathematical mod
  o.w1 = (float)__dsub_rn(gf, g0d);
  o.R2 = R2;
  o.fr = __dsub_rn(q, floor(q));
  o.dx = dx;
  o.dy = dy;
  o.dz = dz;
  return true;
}

// Complex amplitude sqrt(s0dA) G(theta) / R^2 exp(-i 2 pi fr)  (step A5), fp32 from here on.
__device__ __forceinline__ float2 amplitude(const AccParams& p, const Geo& g, float s0dA) {
  const float dx = (float)g.dx, dy = (float)g.dy, dz = (float)g.dz;
  const float inv_R2 = __frcp_rn((float)g.R2);
  const float cx = dy * p.bz - dz * p.by;
  const float cy = dz * p.bx - dx * p.bz;
  const float cz = dx * p.by - dy * p.bx;
  const float sin2 = (cx * cx + cy * cy + cz * cz) * inv_R2;
  const float A = __fsqrt_rn(s0dA) * __expf(-p.alpha * sin2) * inv_R2;
  float ph = (float)g.fr;               // [0,1]
  ph -= (ph >= 0.5f) ? 1.0f : 0.0f;     // [-0.5,0.5): MUFU sin/cos are most accurate near 0
  float sn, cs;
  __sincosf(6.283185307179586f * ph, &sn, &cs);
  return make_float2(A * cs, -A * sn);
}

// ---------------------------------------------------------------------------------------------
// Variant 0: reference kernel.  One scatterer per thread, global fp32x2 reductions into T.
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) acc_reference_kernel(AccParams p) {
  const unsigned long long stride = (unsigned long long)gridDim.x * blockDim.x;
  for (unsigned long long i = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; i < p.n;
       i += stride) {
    const float s0 = p.s0dA[i];
    if (!(s0 > 0.0f)) continue;
    Geo g;
    if (!canonical_geometry(p, p.x[i], p.y[i], p.z[i], p.vx[i], p.vy[i], p.vz[i], g)) continue;
    const float2 c = amplitude(p, g, s0);
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
  for (unsigned long long i = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; i < p.n;
       i += stride) {
    Geo g;
    if (canonical_geometry(p, p.x[i], p.y[i], p.z[i], p.vx[i], p.vy[i], p.vz[i], g)) {
      g0[i] = g.g0;
      k[i] = g.k;
    } else {
      g0[i] = SIM_GATE_NONE;
      k[i] = -1;
    }
  }
}

// ---------------------------------------------------------------------------------------------
// Variant 1: shared-memory tile kernel.
//   * persistent blocks take "super-chunks" of consecutive scatterers from a ticket counter;
//   * each block keeps a window of W Doppler bins x all G gates x R replicas of the spectrum in
//     shared memory (fp32 complex, CAS-add: sm_100a has no native shared fp32 atomic add);
//   * the window follows the data (re-centred per super-chunk, flushed only when it has to move);
//     contributions outside it go straight to T with global fp32x2 reductions;
//   * one flush of the touched window per move / at the end (step A7).
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ void smem_cadd(float2* cell, float2 v) {
  unsigned long long* a = reinterpret_cast<unsigned long long*>(cell);
  unsigned long long old = *a, assumed;
  do {
    assumed = old;
    float2 f;
    f.x = __uint_as_float((unsigned)(assumed & 0xffffffffull)) + v.x;
    f.y = __uint_as_float((unsigned)(assumed >> 32)) + v.y;
    const unsigned long long want =
        (unsigned long long)__float_as_uint(f.x) | ((unsigned long long)__float_as_uint(f.y) << 32);
    old = atomicCAS(a, assumed, want);
  } while (old != assumed);
}

struct TileState {
  int k0;        // first bin of the window
  int valid;     // window has been placed
};

__device__ __forceinline__ void tile_add(const AccParams& p, float2* tile, int k0, int r, int g, int k,
                                         float2 v, unsigned& misses) {
  if ((unsigned)g >= (unsigned)p.G) return;
  const unsigned kw = (unsigned)(k - k0) & (unsigned)(p.N - 1);
  if (kw < (unsigned)p.W) {
    smem_cadd(&tile[((size_t)(g * p.W + (int)kw)) * p.R + r], v);
  } else {
    atomicAdd(&p.T[(size_t)g * p.N + k], v);
    ++misses;
  }
}

__device__ void tile_flush(const AccParams& p, float2* tile, int k0) {
  const int cells = p.G * p.W;
  for (int c = threadIdx.x; c < cells; c += blockDim.x) {
    float2* rep = tile + (size_t)c * p.R;
    float sx = 0.f, sy = 0.f;
    for (int r = 0; r < p.R; ++r) {
      sx += rep[r].x;
      sy += rep[r].y;
      rep[r] = make_float2(0.f, 0.f);
    }
    if (sx != 0.f || sy != 0.f) {
      const int g = c / p.W, kw = c - g * p.W;
      atomicAdd(&p.T[(size_t)g * p.N + ((k0 + kw) & (p.N - 1))], make_float2(sx, sy));
    }
  }
}

__device__ __forceinline__ void process_one(const AccParams& p, float2* tile, int k0, int r, float xf,
                                            float yf, float zf, float vxf, float vyf, float vzf,
                                            float s0, unsigned& misses) {
  if (!(s0 > 0.0f)) return;
  Geo g;
  if (!canonical_geometry(p, xf, yf, zf, vxf, vyf, vzf, g)) return;
  const float2 c = amplitude(p, g, s0);
  const float w1 = g.w1, w0 = 1.0f - w1;
  tile_add(p, tile, k0, r, g.g0, g.k, make_float2(w0 * c.x, w0 * c.y), misses);
  tile_add(p, tile, k0, r, g.g0 + 1, g.k, make_float2(w1 * c.x, w1 * c.y), misses);
}

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

__global__ void __launch_bounds__(kAccThreads, 1) acc_tile_kernel(AccParams p) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  float2* tile = reinterpret_cast<float2*>(smem_raw);
  __shared__ unsigned long long s_ticket;
  __shared__ int s_ref, s_min, s_max, s_k0;

  const int tid = threadIdx.x;
  const int r = tid & (p.R - 1);
  const int cells = p.G * p.W * p.R;
  for (int c = tid; c < cells; c += blockDim.x) tile[c] = make_float2(0.f, 0.f);

  const unsigned long long n_sc = (p.n + p.superchunk - 1) / p.superchunk;
  int k0 = 0;
  bool have_window = false;
  unsigned misses = 0, flushes = 0;

  for (;;) {
    __syncthreads();  // tile zeroed / previous super-chunk finished; s_* free
    if (tid == 0) {
      s_ticket = atomicAdd(&p.counters[kCtrTicket], 1u);
      s_ref = -1;
      s_min = 1 << 30;
      s_max = -(1 << 30);
    }
    __syncthreads();
    const unsigned long long sc = s_ticket;
    if (sc >= n_sc) break;
    const unsigned long long base = sc * p.superchunk;
    const unsigned long long end = (base + p.superchunk < p.n) ? base + p.superchunk : p.n;

    // ---- place the Doppler window from 64 samples spread over the super-chunk ----
    int my_k = -1;
    if (tid < 64) {
      const unsigned long long i = base + (end - base) * (unsigned long long)tid / 64ull;
      Geo g;
      if (canonical_geometry(p, p.x[i], p.y[i], p.z[i], p.vx[i], p.vy[i], p.vz[i], g)) {
        my_k = g.k;
        atomicMax(&s_ref, (tid << 16) | g.k);  // any valid sample serves as the reference bin
      }
    }
    __syncthreads();
    if (s_ref >= 0) {
      const int kr = s_ref & 0xffff;
      if (my_k >= 0) {
        const int d = ((my_k - kr + p.N / 2) & (p.N - 1)) - p.N / 2;  // signed circular offset
        atomicMin(&s_min, d);
        atomicMax(&s_max, d);
      }
      __syncthreads();
      const int centre = kr + (s_min + s_max) / 2;
      const int lo = (centre - p.W / 4 - k0) & (p.N - 1), hi = (centre + p.W / 4 - k0) & (p.N - 1);
      const bool fits = have_window && lo < p.W && hi < p.W && lo <= hi;
      if (!fits) {
        if (have_window) {
          tile_flush(p, tile, k0);
          ++flushes;
        }
        if (tid == 0) s_k0 = (centre - p.W / 2) & (p.N - 1);
        __syncthreads();  // flush done, new origin published
        k0 = s_k0;
        have_window = true;
      }
    }

    // ---- stream the super-chunk: 4 scatterers per thread per chunk, next chunk prefetched ----
    unsigned long long i = base + (unsigned long long)tid * kAccPerThread;
    Quad cur;
    bool cur_full = false;
    if (i + kAccPerThread <= end) {
      load_quad(p, i, cur);
      cur_full = true;
    }
    for (unsigned long long cb = base; cb < end; cb += kAccChunk) {
      const unsigned long long inext = i + kAccChunk;
      Quad nxt;
      bool nxt_full = false;
      if (inext + kAccPerThread <= end) {
        load_quad(p, inext, nxt);
        nxt_full = true;
      }
      if (cur_full) {
        process_one(p, tile, k0, r, cur.x.x, cur.y.x, cur.z.x, cur.vx.x, cur.vy.x, cur.vz.x, cur.s.x, misses);
        process_one(p, tile, k0, r, cur.x.y, cur.y.y, cur.z.y, cur.vx.y, cur.vy.y, cur.vz.y, cur.s.y, misses);
        process_one(p, tile, k0, r, cur.x.z, cur.y.z, cur.z.z, cur.vx.z, cur.vy.z, cur.vz.z, cur.s.z, misses);
        process_one(p, tile, k0, r, cur.x.w, cur.y.w, cur.z.w, cur.vx.w, cur.vy.w, cur.vz.w, cur.s.w, misses);
      } else {
        for (unsigned long long j = i; j < end && j < i + kAccPerThread; ++j)  // ragged tail of the input
          process_one(p, tile, k0, r, p.x[j], p.y[j], p.z[j], p.vx[j], p.vy[j], p.vz[j], p.s0dA[j], misses);
      }
      cur = nxt;
      cur_full = nxt_full;
      i = inext;
    }
  }

  __syncthreads();
  if (have_window) {
    tile_flush(p, tile, k0);
    ++flushes;
  }
  if (misses) atomicAdd(&p.counters[kCtrMiss], misses);
  if (tid == 0 && flushes) atomicAdd(&p.counters[kCtrFlush], flushes);
}

// ---------------------------------------------------------------------------------------------
// Launchers
// ---------------------------------------------------------------------------------------------
cudaError_t acc_tile_smem_bytes(int G, int W, int R, size_t* bytes) {
  *bytes = (size_t)G * W * R * sizeof(float2);
  return cudaSuccess;
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
  size_t smem = 0;
  acc_tile_smem_bytes(p.G, p.W, p.R, &smem);
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
