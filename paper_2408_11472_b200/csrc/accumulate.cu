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

// Steps A2-A4 of one scatterer.  Returns the packed indices (g0 + 1) | (k << 11), or -1 when the scatterer
// touches no gate / is dropped; w1, fr and delta (fp32) are meaningful only for a non-negative code.
//   FAST = false: the canonical sequence for every scatterer.
//   FAST = true:  delta = R - rg0 from u = R^2 - rg0^2 by a 4-term series and 1/R by a 3-term series (no
//   sqrt, no divide), gate and bin read from 2^-20 fixed point; whenever a coordinate lies within `guard`
//   of a boundary the canonical sequence decides (bit-exact indices).
// Written branch-free except for the rare guard-band call.
template <bool FAST>
__device__ __forceinline__ int geometry(const AccParams& p, float xf, float yf, float zf, float vxf,
                                        float vyf, float vzf, float& w1, float& fr, float& delta_f,
                                        unsigned& fallbacks) {
  const double dx = __dsub_rn((double)xf, p.sx);
  const double dy = __dsub_rn((double)yf, p.sy);
  const double dz = __dsub_rn((double)zf, p.sz);
  const double R2 = __fma_rn(dz, dz, __fma_rn(dy, dy, __dmul_rn(dx, dx)));
  if (!FAST) {
    Geo g;
    if (!canonical(p, dx, dy, dz, R2, vxf, vyf, vzf, g)) return -1;
    w1 = g.w1; fr = g.fr; delta_f = g.delta;
    return (g.g0 + 1) | (g.k << 11);
  }
  const double u = (R2 - p.rg0sq_hi) - p.rg0sq_lo;
  const bool inwin = (u >= p.u_lo) && (u <= p.u_hi);  // false: certainly outside the window (or NaN)
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
  const bool near = ((unsigned)(gfrac - p.guard) >= span) | ((unsigned)(kfrac - p.guard) >= span) |
                    !(fabs(kf) < 1024.0);
  if (inwin && near) {  // rare: a coordinate sits in the guard band
    ++fallbacks;
    Geo g;
    if (!canonical(p, dx, dy, dz, R2, vxf, vyf, vzf, g)) return -1;
    w1 = g.w1; fr = g.fr; delta_f = g.delta;
    return (g.g0 + 1) | (g.k << 11);
  }
  const int g0 = gfx >> kFracBits;
  w1 = (float)gfrac * kFxScale;
  fr = phase_fraction(p.two_over_lambda, p.fr0, delta);
  delta_f = (float)gfx * p.dR_fx;
  const bool ok = inwin & (g0 >= -1) & (g0 < p.G);
  return ok ? ((g0 + 1) | (((kfx >> kFracBits) & (p.N - 1)) << 11)) : -1;
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

// fp32 offsets from the satellite (hi + lo split of its position keeps the relative error at 2^-23)
__device__ __forceinline__ void offsets_f32(const AccParams& p, float xf, float yf, float zf, float& dx,
                                            float& dy, float& dz) {
  dx = (xf - p.sxh) - p.sxl;
  dy = (yf - p.syh) - p.syl;
  dz = (zf - p.szh) - p.szl;
}

// Step A5: sqrt(s0dA) G(theta) / R^2 exp(-i 2 pi fr), all fp32.  Returns |c| too.
__device__ __forceinline__ float2 amplitude(const AccParams& p, float dx, float dy, float dz, float delta_f,
                                            float fr, float s0dA, float& A) {
  const float e = delta_f * p.inv_rg0_f;
  const float inv_R2 = p.inv_rg0sq_f * fmaf(e, fmaf(e, 3.0f, -2.0f), 1.0f);  // 1/(rg0 (1+e))^2 to e^3
  const float cx = dy * p.bz - dz * p.by;
  const float cy = dz * p.bx - dx * p.bz;
  const float cz = dx * p.by - dy * p.bx;
  const float sin2 = (cx * cx + cy * cy + cz * cz) * inv_R2;
  A = sqrt_approx(s0dA) * ex2_approx(p.neg_alpha_log2e * sin2) * inv_R2;
  float sn, cs;
  __sincosf(6.283185307179586f * fr, &sn, &cs);
  return make_float2(A * cs, -A * sn);
}

// ---------------------------------------------------------------------------------------------
// Variant 0: reference kernel.  One scatterer per thread, global fp32x2 reductions into T.
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) acc_reference_kernel(AccParams p) {
  const bool fast = p.index_path && p.fast_ok;
  const unsigned long long stride = (unsigned long long)gridDim.x * blockDim.x;
  unsigned fb = 0;
  for (unsigned long long i = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; i < p.n;
       i += stride) {
    const float s0 = p.s0dA[i];
    if (!(s0 > 0.0f)) continue;
    const float xf = p.x[i], yf = p.y[i], zf = p.z[i];
    float w1, fr, df;
    const int code = fast ? geometry<true>(p, xf, yf, zf, p.vx[i], p.vy[i], p.vz[i], w1, fr, df, fb)
                          : geometry<false>(p, xf, yf, zf, p.vx[i], p.vy[i], p.vz[i], w1, fr, df, fb);
    if (code < 0) continue;
    const int g0 = (code & 2047) - 1, k = code >> 11;
    float dx, dy, dz, A;
    offsets_f32(p, xf, yf, zf, dx, dy, dz);
    const float2 c = amplitude(p, dx, dy, dz, df, fr, s0, A);
    const float w0 = 1.0f - w1;
    if (g0 >= 0) atomicAdd(&p.T[(size_t)g0 * p.N + k], make_float2(w0 * c.x, w0 * c.y));
    if (g0 + 1 < p.G) atomicAdd(&p.T[(size_t)(g0 + 1) * p.N + k], make_float2(w1 * c.x, w1 * c.y));
  }
}

// ---------------------------------------------------------------------------------------------
// Index-only kernel (parity pin P11): runs the same index routine as the production kernel.
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) indices_kernel(AccParams p, int32_t* __restrict__ g0,
                                                      int32_t* __restrict__ k) {
  const bool fast = p.index_path && p.fast_ok;
  const unsigned long long stride = (unsigned long long)gridDim.x * blockDim.x;
  unsigned fb = 0;
  for (unsigned long long i = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; i < p.n;
       i += stride) {
    float w1, fr, df;
    const int code = fast ? geometry<true>(p, p.x[i], p.y[i], p.z[i], p.vx[i], p.vy[i], p.vz[i], w1, fr, df, fb)
                          : geometry<false>(p, p.x[i], p.y[i], p.z[i], p.vx[i], p.vy[i], p.vz[i], w1, fr, df, fb);
    g0[i] = code >= 0 ? (code & 2047) - 1 : SIM_GATE_NONE;
    k[i] = code >= 0 ? (code >> 11) : -1;
  }
  if (fb) atomicAdd(&p.counters[kCtrFallback], fb);
}

// ---------------------------------------------------------------------------------------------
// Variant 1: shared-memory tile kernel (the production path).
//
//  * Persistent blocks draw "super-chunks" of consecutive scatterers from a ticket counter and stream them
//    in chunks of CH = 256*PT.  Thread 0 is the scheduler/producer: it moves each chunk's seven 4*CH-byte
//    array slices into a 2-stage shared-memory ring with TMA bulk copies (cp.async.bulk, completion on an
//    mbarrier) two chunks ahead of use -- no registers are held by data in flight, no DRAM latency is
//    exposed at a chunk or super-chunk boundary.
//  * An fp32 pre-test (|u_f32 - u| <= 2^-21 R^2, margin 2^-20 R^2) discards the scatterers that are far
//    outside the gate window before any fp64 work; a warp whose chunk is all outside skips phase 1.
//  * sm_100a has no native shared-memory fp32 atomic add (it is an LDS + ATOMS.CAST.SPIN loop that
//    collapses under the contention of this workload: 10^3..10^4 scatterers per populated cell), but
//    ATOMS.ADD on int32 is native (measured 5 lanes/clk/SM whatever the contention).  Each chunk is
//    therefore one block-floating-point EPOCH:
//      phase 1  geometry + amplitude of the thread's PT scatterers, kept in registers; block statistics
//               (count, mean amplitude, Doppler-offset range, gate range) by REDUX/shuffles + 5 ATOMS;
//      phase 2  the Doppler window [k0, k0+W) is centred on the chunk's own bin range; contributions are
//               scaled by s = 2^e with mean*s in [2^16, 2^17) and added with ATOMS.ADD to an int32 tile
//               [G][W]; a component above 2^20 or a bin outside the window "escapes" to a global fp32x2
//               reduction (exact, rare).  <= 1024 adds of <= 2^20 per cell: no overflow;
//      drain    touched rows of the int tile x 2^-e -> global fp32x2 reductions into T (step A7), tile zeroed.
//    Quantisation: LSB = 2^-e <= mean * 2^-16, so the relative L2 error of an epoch is <= 0.82 * 2^-16
//    = 1.3e-5 whatever the amplitude distribution (mean <= rms); see DESIGN.md.
// ---------------------------------------------------------------------------------------------
namespace sh {  // shared-window addressing (32-bit shared addresses, computed once)
__device__ __forceinline__ unsigned addr(const void* ptr) { return (unsigned)__cvta_generic_to_shared(ptr); }
__device__ __forceinline__ void red_add(unsigned a, int v) {
  asm volatile("red.shared.add.s32 [%0], %1;" ::"r"(a), "r"(v) : "memory");
}
__device__ __forceinline__ void red_min(unsigned a, int v) {
  asm volatile("red.shared.min.s32 [%0], %1;" ::"r"(a), "r"(v) : "memory");
}
__device__ __forceinline__ void red_max(unsigned a, int v) {
  asm volatile("red.shared.max.s32 [%0], %1;" ::"r"(a), "r"(v) : "memory");
}
__device__ __forceinline__ int ld(unsigned a) {
  int v;
  asm volatile("ld.shared.s32 %0, [%1];" : "=r"(v) : "r"(a) : "memory");
  return v;
}
__device__ __forceinline__ float ldf(unsigned a) {
  float v;
  asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(a) : "memory");
  return v;
}
__device__ __forceinline__ void st(unsigned a, int v) {
  asm volatile("st.shared.s32 [%0], %1;" ::"r"(a), "r"(v) : "memory");
}
__device__ __forceinline__ void stf(unsigned a, float v) {
  asm volatile("st.shared.f32 [%0], %1;" ::"r"(a), "f"(v) : "memory");
}
__device__ __forceinline__ int2 ld2(unsigned a) {
  int2 v;
  asm volatile("ld.shared.v2.s32 {%0,%1}, [%2];" : "=r"(v.x), "=r"(v.y) : "r"(a) : "memory");
  return v;
}
__device__ __forceinline__ void st2(unsigned a, int x, int y) {
  asm volatile("st.shared.v2.s32 [%0], {%1,%2};" ::"r"(a), "r"(x), "r"(y) : "memory");
}
template <int PT>
__device__ __forceinline__ void ldv(unsigned a, float (&v)[PT]);
template <>
__device__ __forceinline__ void ldv<4>(unsigned a, float (&v)[4]) {
  asm volatile("ld.shared.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(v[0]), "=f"(v[1]), "=f"(v[2]), "=f"(v[3]) : "r"(a) : "memory");
}
template <>
__device__ __forceinline__ void ldv<2>(unsigned a, float (&v)[2]) {
  asm volatile("ld.shared.v2.f32 {%0,%1}, [%2];" : "=f"(v[0]), "=f"(v[1]) : "r"(a) : "memory");
}
// mbarrier + TMA bulk copy (global -> shared, completion counted in bytes on the mbarrier)
__device__ __forceinline__ void mbar_init(unsigned bar, unsigned count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(unsigned bar, unsigned bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned bar, unsigned parity) {
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "WAIT_%=:\n\t"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
      "@!p bra WAIT_%=;\n\t}" ::"r"(bar), "r"(parity) : "memory");
}
__device__ __forceinline__ void bulk_g2s(unsigned dst, const void* src, unsigned bytes, unsigned bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst),
               "l"(src), "r"(bytes), "r"(bar)
               : "memory");
}
}  // namespace sh

// per-chunk block statistics: 3 rotating sets of 8 ints + kAccWarps floats
enum { kStDmin = 0, kStDmax, kStGmin, kStGmax, kStAnyk, kStCnt, kStInts = 8 };

__device__ __forceinline__ void stats_reset(unsigned a) {
  sh::st(a + 4 * kStDmin, INT_MAX);
  sh::st(a + 4 * kStDmax, INT_MIN);
  sh::st(a + 4 * kStGmin, INT_MAX);
  sh::st(a + 4 * kStGmax, INT_MIN);
  sh::st(a + 4 * kStAnyk, 0);
  sh::st(a + 4 * kStCnt, 0);
}

// Scheduler state of thread 0: the sequence of chunks of this block.
struct Cursor {
  unsigned long long next, end;  // next chunk start, end of the current super-chunk
  bool done;
};

// Thread 0: describe the next chunk of the block's sequence in slot `st` (base, valid count; count 0 = end of
// work) and start its TMA copies.  Floats beyond the last whole group of four are left to the consumers.
template <int CH>
__device__ __forceinline__ void produce_chunk(const AccParams& p, Cursor& c, unsigned long long n_sc,
                                              unsigned stage_smem, unsigned desc, unsigned bar) {
  if (!c.done && c.next >= c.end) {
    const unsigned long long sc = atomicAdd(&p.counters[kCtrTicket], 1u);
    if (sc >= n_sc) {
      c.done = true;
    } else {
      c.next = sc * p.superchunk;
      c.end = (c.next + p.superchunk < p.n) ? c.next + p.superchunk : p.n;
    }
  }
  unsigned nvalid = 0;
  unsigned long long base = 0;
  if (!c.done) {
    base = c.next;
    nvalid = (unsigned)((c.end - base < (unsigned long long)CH) ? c.end - base : CH);
    c.next = base + nvalid;
  }
  asm volatile("st.shared.v2.u32 [%0], {%1,%2};" ::"r"(desc), "r"((unsigned)base), "r"((unsigned)(base >> 32)) : "memory");
  sh::st(desc + 8, (int)nvalid);
  const unsigned bytes = (nvalid & ~3u) * 4u;
  sh::mbar_arrive_expect_tx(bar, 7u * bytes);  // release: the descriptor is visible to whoever sees the phase complete
  if (bytes) {
    const float* src[7] = {p.x, p.y, p.z, p.vx, p.vy, p.vz, p.s0dA};
#pragma unroll
    for (int a = 0; a < 7; ++a) sh::bulk_g2s(stage_smem + (unsigned)a * CH * 4u, src[a] + base, bytes, bar);
  }
}

template <int PT, int MB, bool FAST>
__global__ void __launch_bounds__(kAccThreads, MB) acc_tile_kernel(AccParams p) {
  constexpr int CH = kAccThreads * PT;
  constexpr unsigned kStageBytes = 7u * CH * 4u;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  __shared__ int s_stat[3][kStInts];
  __shared__ float s_wsum[3][kAccWarps];
  __shared__ __align__(8) unsigned long long s_bar[2];
  __shared__ __align__(8) unsigned s_desc[2][4];

  const int cells = p.G * p.W;
  const unsigned stage0 = sh::addr(smem_raw);                 // 2 stages x 7 arrays x CH floats
  const unsigned tile_i = stage0 + 2u * kStageBytes;           // int2 [G][W]
  const unsigned stat0 = sh::addr(&s_stat[0][0]), wsum0 = sh::addr(&s_wsum[0][0]);
  const unsigned bar0 = sh::addr(&s_bar[0]), desc0 = sh::addr(&s_desc[0][0]);

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int N = p.N, W = p.W, halfW = W >> 1, halfN = N >> 1;
  const int logW = 31 - __clz(W);
  for (int c = tid; c < cells; c += kAccThreads) sh::st2(tile_i + 8u * c, 0, 0);
  if (tid < 3) stats_reset(stat0 + 4u * kStInts * tid);
  const unsigned long long n_sc = (p.n + p.superchunk - 1) / p.superchunk;
  Cursor cursor{0, 0, false};
  if (tid == 0) {
    sh::mbar_init(bar0, 1);
    sh::mbar_init(bar0 + 8, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    produce_chunk<CH>(p, cursor, n_sc, stage0, desc0, bar0);
    produce_chunk<CH>(p, cursor, n_sc, stage0 + kStageBytes, desc0 + 16, bar0 + 8);
  }
  __syncthreads();

  int kc = halfN;  // window centre of the previous chunk (reference of the signed circular Doppler offsets)
  unsigned escapes = 0, fallbacks = 0;

  for (unsigned chunk_no = 0;; ++chunk_no) {
    const unsigned stg = chunk_no & 1u;
    const unsigned stage = stage0 + stg * kStageBytes, desc = desc0 + 16u * stg, bar = bar0 + 8u * stg;
    sh::mbar_wait(bar, (chunk_no >> 1) & 1u);
    const unsigned nvalid = (unsigned)sh::ld(desc + 8);
    if (nvalid == 0) break;  // block-uniform: end of work

    // ---- this thread's PT scatterers: shared-memory stage -> registers ----
    float x[PT], y[PT], z[PT], vx[PT], vy[PT], vz[PT], s0[PT];
    const unsigned e0 = (unsigned)tid * PT;
    if (e0 + PT <= (nvalid & ~3u)) {
      const unsigned a = stage + e0 * 4u;
      sh::ldv<PT>(a + 0u * CH * 4u, x);
      sh::ldv<PT>(a + 1u * CH * 4u, y);
      sh::ldv<PT>(a + 2u * CH * 4u, z);
      sh::ldv<PT>(a + 3u * CH * 4u, vx);
      sh::ldv<PT>(a + 4u * CH * 4u, vy);
      sh::ldv<PT>(a + 5u * CH * 4u, vz);
      sh::ldv<PT>(a + 6u * CH * 4u, s0);
    } else {  // ragged end of the input: not covered by the 16-byte bulk copies; s0dA = 0 contributes nothing
      unsigned long long base;
      asm volatile("ld.shared.u64 %0, [%1];" : "=l"(base) : "r"(desc) : "memory");
#pragma unroll
      for (int j = 0; j < PT; ++j) {
        const bool v = e0 + j < nvalid;
        const unsigned long long i = base + e0 + j;
        x[j] = v ? p.x[i] : 0.0f;
        y[j] = v ? p.y[i] : 0.0f;
        z[j] = v ? p.z[i] : 0.0f;
        vx[j] = v ? p.vx[i] : 0.0f;
        vy[j] = v ? p.vy[i] : 0.0f;
        vz[j] = v ? p.vz[i] : 0.0f;
        s0[j] = v ? p.s0dA[i] : 0.0f;
      }
    }

    // ---- phase 1: geometry + amplitude in registers, block statistics ----
    int code[PT];
    float w1[PT], re[PT], im[PT];
    float dxf[PT], dyf[PT], dzf[PT];
    bool maybe = false;
#pragma unroll
    for (int j = 0; j < PT; ++j) {
      offsets_f32(p, x[j], y[j], z[j], dxf[j], dyf[j], dzf[j]);
      const float uf = fmaf(dzf[j], dzf[j], fmaf(dyf[j], dyf[j], dxf[j] * dxf[j])) - p.rg0sq_f;
      // s0dA <= 0 or NaN: dead.  Pre-test: certainly outside the window (NaN position lands here too).
      const bool live_j = (s0[j] > 0.0f) && (!FAST || (uf >= p.uf_lo && uf <= p.uf_hi));
      code[j] = live_j ? 0 : -1;
      maybe |= live_j;
    }
    int cnt = 0, dmin = INT_MAX, dmax = INT_MIN, gmin = INT_MAX, gmax = INT_MIN, anyk = 0;
    float sumA = 0.0f;
    if (__any_sync(0xffffffffu, maybe)) {  // warp-uniform: skip warps that are entirely dark
#pragma unroll
      for (int j = 0; j < PT; ++j) {
        if (code[j] < 0) continue;
        float fr, df;
        code[j] = geometry<FAST>(p, x[j], y[j], z[j], vx[j], vy[j], vz[j], w1[j], fr, df, fallbacks);
        float A;
        const float2 c = amplitude(p, dxf[j], dyf[j], dzf[j], df, fr, s0[j], A);
        re[j] = c.x;
        im[j] = c.y;
        const bool ok = code[j] >= 0;
        const int k = code[j] >> 11, g0 = (code[j] & 2047) - 1;
        const int d = ((k - kc + halfN) & (N - 1)) - halfN;  // signed circular offset from the last centre
        dmin = min(dmin, ok ? d : INT_MAX);
        dmax = max(dmax, ok ? d : INT_MIN);
        gmin = min(gmin, ok ? g0 : INT_MAX);
        gmax = max(gmax, ok ? g0 : INT_MIN);
        anyk = ok ? k : anyk;
        cnt += ok ? 1 : 0;
        sumA += ok ? A : 0.0f;
      }
    }
    const unsigned st = stat0 + 4u * kStInts * (chunk_no % 3u);
    const unsigned wsum = wsum0 + 4u * kAccWarps * (chunk_no % 3u);
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
        sh::red_min(st + 4 * kStDmin, dmin);
        sh::red_max(st + 4 * kStDmax, dmax);
        sh::red_min(st + 4 * kStGmin, gmin);
        sh::red_max(st + 4 * kStGmax, gmax);
        sh::red_add(st + 4 * kStCnt, cnt);
        sh::st(st + 4 * kStAnyk, anyk);
      }
    }
    if (lane == 0) sh::stf(wsum + 4u * warp, live ? sumA : 0.0f);
    __syncthreads();  // (A) statistics complete; stage `stg` fully read; every drain of the previous chunk done
    if (tid == 0) {
      // the set read one chunk ago is next written after the next (A): safe to reset now
      stats_reset(stat0 + 4u * kStInts * ((chunk_no + 2u) % 3u));
      produce_chunk<CH>(p, cursor, n_sc, stage, desc, bar);  // chunk_no + 2 into the stage just consumed
    }

    const int tot = sh::ld(st + 4 * kStCnt);
    if (tot == 0) continue;  // block-uniform: nothing illuminated in this chunk

    // ---- Doppler window of this epoch, centred on the chunk's own bin range ----
    const int bdmin = sh::ld(st + 4 * kStDmin), bdmax = sh::ld(st + 4 * kStDmax);
    if (W < N) kc = ((bdmax - bdmin < W) ? kc + ((bdmin + bdmax + 1) >> 1) : sh::ld(st + 4 * kStAnyk)) & (N - 1);
    const int k0 = (kc - halfW) & (N - 1);

    // ---- block-floating-point scale of this epoch: mean * s in [2^16, 2^17) ----
    float tsum = 0.0f;
#pragma unroll
    for (int w = 0; w < kAccWarps; ++w) tsum += sh::ldf(wsum + 4u * w);
    const float mean = tsum / (float)tot;
    int ex = 16 - (((__float_as_int(mean) >> 23) & 0xff) - 127);
    ex = max(-126, min(127, ex));
    const float s = __int_as_float((ex + 127) << 23);
    const float inv_s = __int_as_float((127 - ex) << 23);
    const float lim = 1048575.0f * inv_s;  // |component| * s <= 2^20 - 1

    // ---- phase 2: native int32 shared-memory atomics ----
    bool esc_any = false;
#pragma unroll
    for (int j = 0; j < PT; ++j) {
      const int k = code[j] >> 11, g0 = (code[j] & 2047) - 1;
      const unsigned kw = (unsigned)(k - k0) & (unsigned)(N - 1);
      const bool ok = code[j] >= 0;
      const bool fits = ok && kw < (unsigned)W && fmaxf(fabsf(re[j]), fabsf(im[j])) <= lim;
      const float w1s = w1[j] * s, w0s = s - w1s;
      // round(v * s) by the 1.5 * 2^23 trick (|v * s| <= 2^20): low mantissa bits, bias removed
      const unsigned a0 = tile_i + 8u * (unsigned)((g0 << logW) + (int)kw);
      if (fits && g0 >= 0) {
        sh::red_add(a0, __float_as_int(fmaf(re[j], w0s, 12582912.0f)) - 0x4B400000);
        sh::red_add(a0 + 4, __float_as_int(fmaf(im[j], w0s, 12582912.0f)) - 0x4B400000);
      }
      if (fits && g0 + 1 < p.G) {
        const unsigned a1 = a0 + 8u * (unsigned)W;
        sh::red_add(a1, __float_as_int(fmaf(re[j], w1s, 12582912.0f)) - 0x4B400000);
        sh::red_add(a1 + 4, __float_as_int(fmaf(im[j], w1s, 12582912.0f)) - 0x4B400000);
      }
      code[j] = (ok && !fits) ? code[j] : -1;  // what is left escapes
      esc_any |= (ok && !fits);
    }
    if (__any_sync(0xffffffffu, esc_any)) {  // rare
#pragma unroll
      for (int j = 0; j < PT; ++j) {
        if (code[j] < 0) continue;
        const int k = code[j] >> 11, g0 = (code[j] & 2047) - 1;
        const float w0 = 1.0f - w1[j];
        if (g0 >= 0) atomicAdd(&p.T[(size_t)g0 * N + k], make_float2(w0 * re[j], w0 * im[j]));
        if (g0 + 1 < p.G) atomicAdd(&p.T[(size_t)(g0 + 1) * N + k], make_float2(w1[j] * re[j], w1[j] * im[j]));
        ++escapes;
      }
    }
    __syncthreads();  // (B) all atomics of the epoch landed

    // ---- drain (step A7): touched rows of the int tile -> global fp32x2 reductions ----
    const int r0 = max(sh::ld(st + 4 * kStGmin), 0), r1 = min(sh::ld(st + 4 * kStGmax) + 1, p.G - 1);
    const int dbase = r0 << logW, dcells = (r1 - r0 + 1) << logW;
    for (int cc = tid; cc < dcells; cc += kAccThreads) {
      const int c = dbase + cc;
      const int2 v = sh::ld2(tile_i + 8u * (unsigned)c);
      if (v.x | v.y) {
        sh::st2(tile_i + 8u * (unsigned)c, 0, 0);
        const int g = c >> logW, kw = c & (W - 1);
        atomicAdd(&p.T[(size_t)g * N + ((k0 + kw) & (N - 1))], make_float2((float)v.x * inv_s, (float)v.y * inv_s));
      }
    }
  }

  if (escapes) atomicAdd(&p.counters[kCtrEscape], escapes);
  if (fallbacks) atomicAdd(&p.counters[kCtrFallback], fallbacks);
}

// ---------------------------------------------------------------------------------------------
// Launchers
// ---------------------------------------------------------------------------------------------
size_t acc_tile_smem_bytes(int G, int W, int per_thread) {
  return (size_t)2 * 7 * kAccThreads * per_thread * sizeof(float) + (size_t)G * W * sizeof(int2);
}

typedef void (*TileKernel)(AccParams);

// (scatterers per thread, resident blocks per SM the register budget is compiled for, index path)
static TileKernel tile_kernel(int per_thread, int min_blocks, bool fast) {
  if (per_thread == 2) {
    if (min_blocks >= 4) return fast ? acc_tile_kernel<2, 4, true> : acc_tile_kernel<2, 4, false>;
    return fast ? acc_tile_kernel<2, 3, true> : acc_tile_kernel<2, 3, false>;
  }
  if (min_blocks >= 3) return fast ? acc_tile_kernel<4, 3, true> : acc_tile_kernel<4, 3, false>;
  return fast ? acc_tile_kernel<4, 2, true> : acc_tile_kernel<4, 2, false>;
}

cudaError_t acc_tile_blocks_per_sm(int G, int W, int per_thread, int min_blocks, int* blocks) {
  const size_t smem = acc_tile_smem_bytes(G, W, per_thread);
  int b = 0;
  *blocks = 1 << 30;
  for (int fast = 0; fast < 2; ++fast) {
    TileKernel k = tile_kernel(per_thread, min_blocks, fast != 0);
    cudaError_t e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&b, k, kAccThreads, smem);
    if (e != cudaSuccess) return e;
    if (b < *blocks) *blocks = b;
  }
  return cudaSuccess;
}

cudaError_t launch_accumulate(const AccParams& p, int variant, int per_thread, int min_blocks, int blocks,
                              cudaStream_t st, int* launches) {
  if (p.n == 0) return cudaSuccess;
  if (variant == 0) {
    unsigned long long want = (p.n + 255) / 256;
    const unsigned long long cap = (unsigned long long)blocks * 8;
    const int grid = (int)(want < cap ? want : cap);
    acc_reference_kernel<<<grid, 256, 0, st>>>(p);
    ++*launches;
    return cudaGetLastError();
  }
  const size_t smem = acc_tile_smem_bytes(p.G, p.W, per_thread);
  cudaError_t e = cudaMemsetAsync(p.counters + kCtrTicket, 0, sizeof(unsigned int), st);
  if (e != cudaSuccess) return e;
  const unsigned long long n_sc = (p.n + p.superchunk - 1) / p.superchunk;
  const int grid = (int)(n_sc < (unsigned long long)blocks ? n_sc : (unsigned long long)blocks);
  tile_kernel(per_thread, min_blocks, p.index_path && p.fast_ok)<<<grid, kAccThreads, smem, st>>>(p);
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
