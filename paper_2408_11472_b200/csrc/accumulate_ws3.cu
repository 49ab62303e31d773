// Steps A1-A7, production kernel v3: scatterers -> spectrum T_u[G][N] (Algorithm 1 body and
// `rasterize`).  sm_100a, no tensor cores: a streaming scan of 28 B per scatterer with a
// scatter-add, bounded by HBM bandwidth, instruction issue and the shared-memory atomic unit.
//
// Same method as accumulate_ws.cu (TMA stage ring, block-floating int32 tiles, per-epoch drain); what changed
// after the v2 profile (profiles/r01_v2_ws_kernel.md):
//   * three roles instead of two: warps 0..NCW-1 compute (NCW a multiple of 4: the same number on every SM
//     sub-partition), warp NCW only PRODUCES (ticket counter -> TMA bulk copies, next ticket prefetched), warp
//     NCW+1 only DRAINS finished tiles (step A7); both sleep in hardware-suspended mbarrier waits.  A drain no longer delays
//     the next loads;
//   * the two control warps wait with a suspend-time hint (v2 spent 20 % of its issue slots spinning); the block's
//     end is signalled through the barriers themselves (the compute warps publish the index of the final epoch);
//   * the tile has one padding row below gate 0 and one above gate G-1, so the two gate halves need no
//     per-half bounds predicate; the drain warp scans every row (tracking the touched rows cost the compute warps
//     more than the scan costs the drain warp);
//   * 8 compute warps with 96 registers each, 4 scatterers per lane per chunk, all four in flight together;
//   * the polynomial index path runs straight through for the scatterers in flight and ONE cold block per group
//     re-decides the rare guard-band cases: a call site in the hot flow cuts the live ranges of ~40 constants;
//   * long fixed-point epochs (8191 scatterers by default) with an admitted magnitude range that shrinks as the
//     epoch grows, so that no cell can overflow: every epoch boundary is a rendez-vous of the block's warps;
//   * scheduling units are visited in a scattered order (golden-ratio stride), so that dark parts of the scene
//     (DRAM-bound) and illuminated parts (issue-bound) are in flight at the same time.
// Measurements and the experiments behind each choice: profiles/r01_v3_ws3_kernel.md, profiles/r01_v3_final.md.
#include <climits>

#include "ptx_util.cuh"
#include "scatter_math.cuh"

namespace simk {

constexpr int kW3MaxStages = 6;

// epoch parameter slot (ring of 4): state, first bin of the Doppler window, scale exponent
enum { kS3State = 0, kS3K0 = 1, kS3Ex = 2, kS3Ints = 4 };
enum { kT3Unset = 0, kT3Claimed = 1, kT3Ready = 2 };

int acc_ws3_chunk(int ncw, int pt) { return ncw * 32 * pt; }

size_t acc_ws3_smem_bytes(int G, int W, int ncw, int pt, int stages) {
  const size_t tiles = (G > 0) ? (size_t)2 * 2 * (G + 2) * (W + 1) * sizeof(int) : 0;
  return (size_t)stages * 7 * acc_ws3_chunk(ncw, pt) * sizeof(float) + tiles;
}

// Scheduler state of the producer's lane 0: the sequence of chunks of this block.
struct Cursor3 {
  unsigned long long next, end;   // next chunk start, end of the current super-chunk
  unsigned long long ticket;      // prefetched ticket of the following super-chunk
  bool done;
};

template <int CH>
__device__ __forceinline__ unsigned produce_chunk3(const AccParams& p, Cursor3& c, unsigned long long n_sc,
                                                   unsigned stage_smem, unsigned desc, unsigned bar) {
  if (!c.done && c.next >= c.end) {
    const unsigned long long sc = c.ticket;
    if (sc >= n_sc) {
      c.done = true;
    } else {
      c.next = ((sc * p.sc_stride) % n_sc) * p.superchunk;   // tickets visit the scene in a scattered order
      c.end = (c.next + p.superchunk < p.n) ? c.next + p.superchunk : p.n;
      c.ticket = atomicAdd(&p.counters[kCtrTicket], 1u);   // consumed one super-chunk later: latency hidden
    }
  }
  unsigned nvalid = 0;
  unsigned long long base = 0;
  if (!c.done) {
    base = c.next;
    nvalid = (unsigned)((c.end - base < (unsigned long long)CH) ? c.end - base : CH);
    c.next = base + nvalid;
  }
  sh::st64(desc, base);
  sh::st(desc + 8, (int)nvalid);
  const unsigned bytes = (nvalid & ~3u) * 4u;
  sh::mbar_arrive_expect_tx(bar, 7u * bytes);  // release: the descriptor is visible to whoever sees the phase complete
  if (bytes) {
    const float* src[7] = {p.x, p.y, p.z, p.vx, p.vy, p.vz, p.s0dA};
#pragma unroll
    for (int a = 0; a < 7; ++a) sh::bulk_g2s(stage_smem + (unsigned)a * CH * 4u, src[a] + base, bytes, bar);
  }
  return nvalid;
}

// round(a * b) for |a b| <= 2^22 by the 1.5 * 2^23 trick (round to nearest even: unbiased), as an int
__device__ __forceinline__ int fx_round3(float a, float b) {
  return __float_as_int(fmaf(a, b, 12582912.0f)) - 0x4B400000;
}

__device__ __forceinline__ void wait3(unsigned bar, unsigned parity, unsigned hint_ns) {
  if (hint_ns) sh::mbar_wait_sleepy(bar, parity, hint_ns);
  else sh::mbar_wait(bar, parity);
}

template <int PT>
struct Vec;
template <>
struct Vec<2> {
  float v[2];
  __device__ __forceinline__ void load(unsigned a) {
    const float2 t = sh::ldf2(a);
    v[0] = t.x; v[1] = t.y;
  }
};
template <>
struct Vec<4> {
  float v[4];
  __device__ __forceinline__ void load(unsigned a) {
    const float4 t = sh::ldf4(a);
    v[0] = t.x; v[1] = t.y; v[2] = t.z; v[3] = t.w;
  }
};

template <int NCW, int PT, int IL, int MODE>
__global__ void __launch_bounds__((NCW + 2) * 32, (NCW <= 4 ? 3 : NCW <= 14 ? 2 : 1)) acc_ws3_kernel(AccParams p) {
  constexpr int CH = NCW * 32 * PT;
  constexpr unsigned kStageBytes = 7u * CH * 4u;
  constexpr unsigned kFull = 0xffffffffu;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  __shared__ __align__(8) unsigned long long s_full[kW3MaxStages], s_empty[kW3MaxStages], s_tdone[2], s_tfree[2];
  __shared__ __align__(16) unsigned s_desc[kW3MaxStages][4];
  __shared__ int s_slot[4][kS3Ints];
  __shared__ unsigned s_last;   // index of the block's final epoch, written by the compute warps when they see the end marker

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int S = p.stages, EC = p.epoch_chunks;
  const int G = p.G, N = p.N, W = p.W, RS = W + 1;
  const unsigned stage0 = sh::addr(smem_raw);
  const unsigned tile0 = stage0 + (unsigned)S * kStageBytes;     // int [2 tiles][2 planes: re, im][G + 2][W + 1]
  const unsigned plane_bytes = (unsigned)((G + 2) * RS) * 4u, tile_bytes = 2u * plane_bytes;
  const unsigned full0 = sh::addr(&s_full[0]), empty0 = sh::addr(&s_empty[0]);
  const unsigned tdone0 = sh::addr(&s_tdone[0]), tfree0 = sh::addr(&s_tfree[0]);
  const unsigned desc0 = sh::addr(&s_desc[0][0]), slot0 = sh::addr(&s_slot[0][0]);
  const unsigned last_a = sh::addr(&s_last);

  for (unsigned a = 4u * tid; a < 2u * tile_bytes; a += 4u * (NCW + 2) * 32) sh::st(tile0 + a, 0);
  if (tid < 4) sh::st(slot0 + 4u * kS3Ints * tid + 4 * kS3State, kT3Unset);
  if (tid == 0) {
    sh::st(last_a, (int)kFull);
    for (int s = 0; s < S; ++s) {
      sh::mbar_init(full0 + 8u * s, 1);
      sh::mbar_init(empty0 + 8u * s, NCW);
    }
    for (int b = 0; b < 2; ++b) {
      sh::mbar_init(tdone0 + 8u * b, NCW);
      sh::mbar_init(tfree0 + 8u * b, 1);
    }
    sh::mbar_fence_init();
  }
  __syncthreads();   // the only block-wide barrier

  if (warp == NCW) {
    // ================= producer warp (one lane): ticket counter -> TMA bulk copies =================
    if (lane != 0) return;
    const unsigned long long n_sc = (p.n + p.superchunk - 1) / p.superchunk;
    Cursor3 cur{0, 0, atomicAdd(&p.counters[kCtrTicket], 1u), false};
    unsigned stg = 0, ph = 0;
    for (unsigned c = 0;; ++c) {
      // chunk c - S pulled out of the stage.  Suspended wait: this lane shares an SM sub-partition with compute warps
      if (c >= (unsigned)S) sh::mbar_wait_sleepy(empty0 + 8u * stg, ph ^ 1u, 100000u);
      const unsigned nv = produce_chunk3<CH>(p, cur, n_sc, stage0 + stg * kStageBytes, desc0 + 16u * stg, full0 + 8u * stg);
      if (nv == 0) return;   // the end marker is out
      if (++stg == (unsigned)S) { stg = 0; ph ^= 1u; }
    }
  }

  if (warp == NCW + 1) {
    // ================= drain warp: tile of epoch e -> T (step A7), tile handed back =================
    const int logW = W > 1 ? 32 - __clz(W - 1) : 0, Wp = 1 << logW;   // window rounded up to a power of two: lanes kw >= W idle
    for (unsigned e = 0;; ++e) {
      const unsigned b = e & 1u;
      sh::mbar_wait_sleepy(tdone0 + 8u * b, (e >> 1) & 1u, 100000u);   // every compute warp finished epoch e
      const unsigned slot = slot0 + 4u * kS3Ints * (e & 3u);
      if (sh::ld(slot + 4 * kS3State) == kT3Ready) {
        const int k0 = sh::ld(slot + 4 * kS3K0), ex = sh::ld(slot + 4 * kS3Ex);
        const float inv_s = __int_as_float((127 - ex) << 23);
        const int r0 = 0, r1 = G - 1;   // every row: tracking the touched rows costs the compute warps more than the scan costs here
        const int ncell = (r1 - r0 + 1) << logW;
        const unsigned tile = tile0 + b * tile_bytes;
        // four cells per lane per pass, their eight loads in flight together: the drain must be well under one
        // epoch long or the compute warps wait for their tile (profiles/r01_v3_final.md)
        for (int cc0 = lane; cc0 < ncell; cc0 += 128) {
          int re[4], im[4];
          unsigned a[4];
  #pragma unroll
          for (int u = 0; u < 4; ++u) {
            const int cc = cc0 + 32 * u;
            const int r = r0 + (cc >> logW), kw = cc & (Wp - 1);
            const bool v = cc < ncell && kw < W;
            a[u] = tile + 4u * (unsigned)((r + 1) * RS + kw);
            re[u] = v ? sh::ld(a[u]) : 0;
            im[u] = v ? sh::ld(a[u] + plane_bytes) : 0;
          }
  #pragma unroll
          for (int u = 0; u < 4; ++u) {
            if (re[u] | im[u]) {
              const int cc = cc0 + 32 * u;
              const int r = r0 + (cc >> logW), kw = cc & (Wp - 1);
              sh::st(a[u], 0);
              sh::st(a[u] + plane_bytes, 0);
              atomicAdd(&p.T[(size_t)r * N + ((k0 + kw) & (N - 1))], make_float2((float)re[u] * inv_s, (float)im[u] * inv_s));
            }
          }
        }
        __syncwarp();
        if (lane == 0) sh::st(slot + 4 * kS3State, kT3Unset);
      }
      __syncwarp();
      if (lane == 0) sh::mbar_arrive(tfree0 + 8u * b);  // release: zeroed tile and reset slot are visible
      if ((unsigned)sh::ld(last_a) == e) return;        // written before the last arrival on tdone of epoch e
    }
  }

  // ================= compute warps =================
  const unsigned e0 = (unsigned)(warp * 32 + lane) * PT;   // this lane's first scatterer in a chunk
  const int halfN = N >> 1;
  unsigned stg = 0, ph = 0;
  unsigned escapes = 0, fallbacks = 0;
  bool more = true;
  const unsigned fx_span = (unsigned)(p.fx_cap - 11) << 23;   // admitted |c| s: [2^11, 2^fx_cap]

  for (unsigned e = 0; more; ++e) {
    const unsigned tile_b = tile0 + (e & 1u) * tile_bytes;
    const unsigned slot = slot0 + 4u * kS3Ints * (e & 3u);
    if (e >= 2) wait3(tfree0 + 8u * (e & 1u), ((e >> 1) - 1u) & 1u, p.wait_hint);  // tile of epoch e-2 drained
    bool have = false;         // this warp holds the epoch's parameters
    int k0 = 0, lo_bits = 0;
    float s = 0.0f;
    int ci = 0;
    for (; ci < EC; ++ci) {
      wait3(full0 + 8u * stg, ph, p.wait_hint);
      const unsigned desc = desc0 + 16u * stg;
      const unsigned nvalid = (unsigned)sh::ld(desc + 8);
      if (nvalid == 0) { more = false; break; }   // block-uniform: end of work

      // ---- step A1: this lane's PT scatterers, shared-memory stage -> registers; stage released at once ----
      Vec<PT> x, y, z, vx, vy, vz, s0;
      if (e0 + PT <= (nvalid & ~3u)) {
        const unsigned a = stage0 + stg * kStageBytes + e0 * 4u;
        x.load(a + 0u * CH * 4u);
        y.load(a + 1u * CH * 4u);
        z.load(a + 2u * CH * 4u);
        vx.load(a + 3u * CH * 4u);
        vy.load(a + 4u * CH * 4u);
        vz.load(a + 5u * CH * 4u);
        s0.load(a + 6u * CH * 4u);
      } else {  // ragged end of the input: not covered by the 16-byte bulk copies; s0dA = 0 contributes nothing
        const unsigned long long base = sh::ld64(desc);
#pragma unroll
        for (int j = 0; j < PT; ++j) {
          const bool v = e0 + j < nvalid;
          const unsigned long long i = base + e0 + j;
          x.v[j] = v ? p.x[i] : 0.0f;
          y.v[j] = v ? p.y[i] : 0.0f;
          z.v[j] = v ? p.z[i] : 0.0f;
          vx.v[j] = v ? p.vx[i] : 0.0f;
          vy.v[j] = v ? p.vy[i] : 0.0f;
          vz.v[j] = v ? p.vz[i] : 0.0f;
          s0.v[j] = v ? p.s0dA[i] : 0.0f;
        }
      }
      __syncwarp();
      if (lane == 0) sh::mbar_arrive(empty0 + 8u * stg);
      if (++stg == (unsigned)S) { stg = 0; ph ^= 1u; }

#pragma unroll
      for (int gi = 0; gi < PT; gi += IL) {   // IL scatterers in flight per lane at a time
        // ---- steps A2-A5 ----
        bool ok[IL];
        Pre q[IL];
        bool any = false;
  #pragma unroll
        for (int j = 0; j < IL; ++j) {
          ok[j] = s0.v[gi + j] > 0.0f;   // s0dA <= 0 or NaN: dead
          q[j] = pre_part<MODE>(p, x.v[gi + j], y.v[gi + j], z.v[gi + j], ok[j]);
          any |= ok[j];
        }
        if (!__any_sync(kFull, any)) continue;   // warp-uniform: the whole warp is dark
        Idx ix[IL];
        float2 c[IL];
        int ab[IL];
        any = false;
        if (MODE == kIdxCanonical) {
  #pragma unroll
          for (int j = 0; j < IL; ++j) {
            ok[j] = index_part<MODE>(p, q[j], vx.v[gi + j], vy.v[gi + j], vz.v[gi + j], ok[j], ix[j], fallbacks);
            float A;
            c[j] = amplitude(p, x.v[gi + j], y.v[gi + j], z.v[gi + j], ix[j].gfx, ix[j].fr, s0.v[gi + j], A);
            ab[j] = __float_as_int(A);
            any |= ok[j];
          }
        } else {
          // polynomial path straight through for all IL scatterers (no call site in the hot flow: calls cut the live
          // ranges of the constants), then ONE cold patch-up for the rare guard-band cases
          bool near[IL], any_near = false;
  #pragma unroll
          for (int j = 0; j < IL; ++j) {
            ok[j] = index_fast<MODE>(p, q[j], vx.v[gi + j], vy.v[gi + j], vz.v[gi + j], ok[j], ix[j], near[j]);
            float A;
            c[j] = amplitude(p, x.v[gi + j], y.v[gi + j], z.v[gi + j], ix[j].gfx, ix[j].fr, s0.v[gi + j], A);
            ab[j] = __float_as_int(A);
            any_near |= near[j];
          }
          if (__any_sync(kFull, any_near)) {
  #pragma unroll
            for (int j = 0; j < IL; ++j) {
              if (near[j]) {
                ++fallbacks;
                // offsets recomputed here (three subtractions) rather than kept alive across the amplitude for this rare case
                ok[j] = canonical(p, __dsub_rn((double)x.v[gi + j], p.sx), __dsub_rn((double)y.v[gi + j], p.sy),
                                  __dsub_rn((double)z.v[gi + j], p.sz), vx.v[gi + j], vy.v[gi + j], vz.v[gi + j], ix[j]);
                float A;
                c[j] = amplitude(p, x.v[gi + j], y.v[gi + j], z.v[gi + j], ix[j].gfx, ix[j].fr, s0.v[gi + j], A);
                ab[j] = __float_as_int(A);
              }
            }
          }
  #pragma unroll
          for (int j = 0; j < IL; ++j) any |= ok[j];
        }
        const unsigned okm = __ballot_sync(kFull, any);
        if (okm == 0) continue;

        // ---- epoch parameters: the first warp with something to add decides them ----
        if (!have) {
          int st = 0;
          if (lane == 0) {
            st = sh::ld_acquire(slot + 4 * kS3State);
            if (st != kT3Ready) st = sh::cas(slot + 4 * kS3State, kT3Unset, kT3Claimed);
          }
          st = __shfl_sync(kFull, st, 0);
          if (st == kT3Unset) {  // this warp won the claim: window and scale from its own scatterers
            int kk = 0;
  #pragma unroll
            for (int j = IL - 1; j >= 0; --j) kk = ok[j] ? ix[j].k : kk;
            const int kref = __shfl_sync(kFull, kk, __ffs(okm) - 1) & (N - 1);
            int dmin = INT_MAX, dmax = INT_MIN, cnt = 0, slog = 0;
  #pragma unroll
            for (int j = 0; j < IL; ++j) {
              const int d = ((ix[j].k - kref + halfN) & (N - 1)) - halfN;   // signed circular bin offset
              dmin = min(dmin, ok[j] ? d : INT_MAX);
              dmax = max(dmax, ok[j] ? d : INT_MIN);
              cnt += ok[j] ? 1 : 0;
              slog += ok[j] ? (ab[j] >> 16) : 0;                            // log2 amplitude, 2^-7 units
            }
            dmin = __reduce_min_sync(kFull, dmin);
            dmax = __reduce_max_sync(kFull, dmax);
            cnt = __reduce_add_sync(kFull, cnt);
            slog = __reduce_add_sync(kFull, slog);
            if (lane == 0) {
              const int centre = (dmax - dmin < W) ? kref + ((dmin + dmax + 1) >> 1) : kref;
              const int E = (slog / cnt) >> 7;                      // biased exponent of the geometric mean
              const int ex = max(-100, min(120, p.fx_target - (E - 127)));   // gmean * 2^ex in [2^16, 2^17) (default)
              sh::st(slot + 4 * kS3K0, (centre - (W >> 1)) & (N - 1));
              sh::st(slot + 4 * kS3Ex, ex);
              sh::st_release(slot + 4 * kS3State, kT3Ready);
            }
            __syncwarp();
          } else if (st == kT3Claimed) {
            while (sh::ld_acquire(slot + 4 * kS3State) != kT3Ready) {
            }
          }
          k0 = sh::ld(slot + 4 * kS3K0);
          const int ex = sh::ld(slot + 4 * kS3Ex);
          s = __int_as_float((ex + 127) << 23);
          lo_bits = (11 - ex + 127) << 23;                    // bits of 2^11 / s
          have = true;
        }

        // ---- step A6: native int32 shared-memory atomics; what does not fit escapes to global fp32 ----
        bool esc_any = false;
        bool esc[IL];
  #pragma unroll
        for (int j = 0; j < IL; ++j) {
          const unsigned kw = (unsigned)(ix[j].k - k0) & (unsigned)(N - 1);
          const bool fits = ok[j] && kw < (unsigned)W && (unsigned)(ab[j] - lo_bits) <= fx_span;
          const float w1s = ix[j].w1 * s, w0s = s - w1s;
          const unsigned a0 = tile_b + 4u * (unsigned)((ix[j].g0 + 1) * RS + (int)kw);   // row g0 (padded by one)
          if (fits) {
            sh::red_add(a0, fx_round3(c[j].x, w0s));
            sh::red_add(a0 + plane_bytes, fx_round3(c[j].y, w0s));
            sh::red_add(a0 + 4u * (unsigned)RS, fx_round3(c[j].x, w1s));
            sh::red_add(a0 + 4u * (unsigned)RS + plane_bytes, fx_round3(c[j].y, w1s));
          }
          esc[j] = ok[j] && !fits;
          esc_any |= esc[j];
        }
        if (__any_sync(kFull, esc_any)) {  // rare
  #pragma unroll
          for (int j = 0; j < IL; ++j) {
            if (esc[j]) {
              const int k = ix[j].k & (N - 1), g0 = ix[j].g0;
              const float w1 = ix[j].w1, w0 = 1.0f - w1;
              if (g0 >= 0) atomicAdd(&p.T[(size_t)g0 * N + k], make_float2(w0 * c[j].x, w0 * c[j].y));
              if (g0 + 1 < G) atomicAdd(&p.T[(size_t)(g0 + 1) * N + k], make_float2(w1 * c[j].x, w1 * c[j].y));
              ++escapes;
            }
          }
        }
      }
    }

    // ---- end of an epoch (or of the input inside one): tile to the drain warp ----
    {
      if (!more && lane == 0) sh::st(last_a, (int)e);   // the final epoch (possibly empty): the drain warp stops after it
      __syncwarp();
      if (lane == 0) sh::mbar_arrive(tdone0 + 8u * (e & 1u));
    }
  }
  if (escapes) atomicAdd(&p.counters[kCtrEscape], escapes);
  if (fallbacks) atomicAdd(&p.counters[kCtrFallback], fallbacks);
}

// Which index routine a launch uses: the polynomial path of the configured Doppler source when the host found
// its error bounds covered by the guard band, else the canonical sequence everywhere.
int acc_index_mode(const AccParams& p);   // accumulate.cu

// ---------------------------------------------------------------------------------------------
// Index-only kernel (parity pin P11, sim_debug_indices): the index routine of the production kernel
// (pre_part + index_part of scatter_math.cuh), one scatterer per thread, s0dA not consulted.
// ---------------------------------------------------------------------------------------------
template <int MODE>
__global__ void __launch_bounds__(256) indices3_kernel(AccParams p, int32_t* __restrict__ g0, int32_t* __restrict__ k) {
  const unsigned long long stride = (unsigned long long)gridDim.x * blockDim.x;
  unsigned fb = 0;
  for (unsigned long long i = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; i < p.n; i += stride) {
    bool live = true;
    const Pre q = pre_part<MODE>(p, p.x[i], p.y[i], p.z[i], live);
    Idx ix;
    const bool ok = index_part<MODE>(p, q, p.vx[i], p.vy[i], p.vz[i], live, ix, fb);
    g0[i] = ok ? ix.g0 : SIM_GATE_NONE;
    k[i] = ok ? (ix.k & (p.N - 1)) : -1;
  }
  if (fb) atomicAdd(&p.counters[kCtrFallback], fb);
}

cudaError_t launch_indices3(const AccParams& p, int32_t* g0, int32_t* k, int sm_count, cudaStream_t st, int* launches) {
  if (p.n == 0) return cudaSuccess;
  const unsigned long long want = (p.n + 255) / 256, cap = (unsigned long long)sm_count * 16;
  const int grid = (int)(want < cap ? want : cap);
  switch (acc_index_mode(p)) {
    case kIdxFast: indices3_kernel<kIdxFast><<<grid, 256, 0, st>>>(p, g0, k); break;
    case kIdxFastPulsePair: indices3_kernel<kIdxFastPulsePair><<<grid, 256, 0, st>>>(p, g0, k); break;
    default: indices3_kernel<kIdxCanonical><<<grid, 256, 0, st>>>(p, g0, k); break;
  }
  ++*launches;
  return cudaGetLastError();
}

// ---------------------------------------------------------------------------------------------
// Launchers
// ---------------------------------------------------------------------------------------------
typedef void (*W3Kernel)(AccParams);

static W3Kernel ws3_kernel(int ncw, int pt, int il, int mode) {
#define W3_CASE(NCW_, PT_, IL_) \
  if (ncw == NCW_ && pt == PT_ && il == IL_)                                                  \
    return mode == kIdxFast ? acc_ws3_kernel<NCW_, PT_, IL_, kIdxFast>                         \
         : mode == kIdxFastPulsePair ? acc_ws3_kernel<NCW_, PT_, IL_, kIdxFastPulsePair>       \
                                     : acc_ws3_kernel<NCW_, PT_, IL_, kIdxCanonical>;
  W3_CASE(8, 2, 2) W3_CASE(8, 4, 4) W3_CASE(8, 4, 2) W3_CASE(12, 2, 2) W3_CASE(16, 4, 2) W3_CASE(20, 4, 2)
#undef W3_CASE
  return nullptr;
}

bool acc_ws3_supported(int ncw, int pt, int il) { return ws3_kernel(ncw, pt, il, kIdxFast) != nullptr; }

cudaError_t acc_ws3_blocks_per_sm(int G, int W, int ncw, int pt, int il, int stages, int* blocks) {
  const size_t smem = acc_ws3_smem_bytes(G, W, ncw, pt, stages);
  *blocks = 1 << 30;
  for (int mode = 0; mode < 3; ++mode) {
    W3Kernel k = ws3_kernel(ncw, pt, il, mode);
    if (!k) return cudaErrorInvalidValue;
    cudaError_t e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    int b = 0;
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&b, k, (ncw + 2) * 32, smem);
    if (e != cudaSuccess) return e;
    if (b < *blocks) *blocks = b;
  }
  return cudaSuccess;
}

cudaError_t launch_accumulate_ws3(const AccParams& p, int ncw, int pt, int il, int blocks, cudaStream_t st, int* launches) {
  if (p.n == 0) return cudaSuccess;
  const int mode = acc_index_mode(p);
  // the canonical-everywhere path calls the out-of-line sequence once per scatterer: two in flight per lane are enough
  if (mode == kIdxCanonical && il == 4 && ws3_kernel(ncw, pt, 2, mode)) il = 2;
  W3Kernel k = ws3_kernel(ncw, pt, il, mode);
  if (!k) return cudaErrorInvalidValue;
  const size_t smem = acc_ws3_smem_bytes(p.G, p.W, ncw, pt, p.stages);
  // per launch: the limit is per function and per device, another handle may have set it for a smaller shape
  cudaError_t e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return e;
  e = cudaMemsetAsync(p.counters + kCtrTicket, 0, sizeof(unsigned int), st);
  if (e != cudaSuccess) return e;
  const unsigned long long n_sc = (p.n + p.superchunk - 1) / p.superchunk;
  const int grid = (int)(n_sc < (unsigned long long)blocks ? n_sc : (unsigned long long)blocks);
  k<<<grid, (ncw + 2) * 32, smem, st>>>(p);
  ++*launches;
  return cudaGetLastError();
}

}  // namespace simk
