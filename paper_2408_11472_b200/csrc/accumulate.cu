// Steps A1-A7: scatterers -> spectrum T_u[G][N] (Algorithm 1 body and `rasterize`).
// sm_100a, no tensor cores: a streaming scan of 28 B per scatterer with a scatter-add, bounded by HBM bandwidth,
// instruction issue and the shared-memory atomic unit.
//
// Production kernel `acc_kernel` (variant 4).  Persistent blocks, two per SM, NCW = 8 warps that all compute (up to 128
// registers per thread):
//   * scheduling units of consecutive scatterers (whole fixed-point epochs) are drawn from a global ticket counter
//     (visited in a scattered order so that dark and illuminated parts of the scene are in flight together) and streamed
//     in chunks of CH = NCW*32*PT through a two-stage shared-memory ring by per-lane 16-byte asynchronous copies
//     (cp.async.cg, LDGSTS: a warp instruction moves 512 contiguous bytes of one array).  There is no producer warp and no
//     hand-shake between warps on the load side: every lane copies exactly the 7 x 16 bytes it will read itself, one chunk
//     ahead, and waits for its own commit group.  (Round 1 used TMA bulk copies issued by a producer warp; per-warp bulk
//     copies and plain ld.global.nc prefetch into registers were measured this round and lost: DESIGN.md section 6.)
//     The units (start, end) sit in a small shared-memory table that the first warp into unit u extends by unit u + 2;
//     a partial unit (ragged end of the input) ends its epoch early;
//   * steps A2-A5 run in registers for IL scatterers at a time: range, gate and Doppler coordinates and the phase in fp64
//     (polynomials in u = R^2 - rg0^2), amplitude in packed fp32 (fma/mul.rn.f32x2: two scatterers per instruction); gate,
//     bin and the guard-band test are derived last, from two fixed-point integers; the rare cases go through ONE cold
//     block per group: guard-band cases are decided by the canonical fp64 sequence, window and range escapes keep their
//     indices and go to the global accumulator;
//   * step A6 is block floating point: native int32 shared-memory reductions (red.shared.add.s32) of round(w c s) into a
//     tile of FOUR planes [lower-gate half | upper-gate half] x [re | im], each [G+1][RS]; s is a power of two fixed per
//     epoch of <= 8191 scatterers from the geometric mean of the first warp's amplitudes, so that no cell can overflow.
//     3 000-20 000 scatterers land in each hot cell and a warp's 32 scatterers hit only ~9 distinct cells, so same-address
//     and same-bank replays are what the atomic unit spends its time on; the four values of a scatterer are therefore
//     issued in a lane-dependent order (lane bit 0 swaps re/im, lane bit 1 swaps lower/upper) and rows and planes are
//     padded (acc_row_stride, acc_plane_words below): 4.1 wavefronts per reduction instruction instead of 9.4;
//   * when the last warp has finished an epoch (an mbarrier phase per tile), every warp drains ITS SHARE of that epoch's
//     gate rows into fp64 global reductions (step A7) at its next chunk boundary, while the second tile already fills
//     with the next epoch: no drain warp, no rendez-vous; a warp that runs ahead sleeps on the mbarrier.  The global
//     accumulator is an fp64 grid (exact enough that 10^5 identical escapes into one cell lose nothing);
//     `acc_finalize_kernel` rounds it to the complex64 spectrum and re-zeroes it.
// Reference kernel `acc_reference_kernel` (variant 0): one thread per scatterer, canonical sequence, global fp64
// reductions; the A/B partner of the production kernel in the parity tests.
// `sim_debug_indices` runs the production kernel itself with DBG = true (same index flow, indices written instead of
// amplitudes accumulated).
#include <climits>
#include <cstdlib>

#include "ptx_util.cuh"
#include "scatter_math.cuh"

namespace simk {

constexpr int kRing = 128;   // chunk table entries: more than two epochs (<= 2 * 31 chunks) + the stage ring

// epoch parameter slot (ring of 4): state, first bin of the Doppler window (unwrapped), scale exponent
enum { kSlotState = 0, kSlotK0 = 1, kSlotEx = 2, kSlotInts = 4 };
enum { kSlotUnset = 0, kSlotClaimed = 1, kSlotReady = 2 };
// scheduling-unit table in shared memory (ring): first scatterer, end, sequence number (= unit index + 1 once published)
int acc_chunk(int ncw, int pt) { return ncw * 32 * pt; }

// Tile layout (bank behaviour simulated on the nadir and PM scenes and confirmed by ncu, profiles/): words per row = 4
// mod 8 (rows g .. g + 7 of one bin then sit in eight different banks), words per plane = 2 mod 32 (the four planes
// that the lanes of one reduction instruction are spread over do not alias bank for bank): 4.1 wavefronts per
// reduction instruction on the white-noise scene against 7.2 for rows of 12 and planes of 12 mod 32, and 9.4 without
// the lane rotation.
int acc_row_stride(int W) {
  int rs = (W + 1) & ~1;
  while ((rs & 7) != 4) rs += 2;
  return rs;
}
// Rows of a plane: G + 1 gate rows, then enough rows to give every lane of a warp its own "dump" word, where the
// reductions of a scatterer that the tile cannot take are sent (never read, never zeroed): the four reductions are
// issued unconditionally, without a branch around them.
static int acc_dump_rows(int W) { return (32 + acc_row_stride(W) - 1) / acc_row_stride(W); }
int acc_plane_words(int G, int W) {
  int w = (G + 1 + acc_dump_rows(W)) * acc_row_stride(W);
  while ((w & 31) != 2) w += 2;
  return w;
}

size_t acc_tile_bytes(int G, int W) { return (size_t)4 * acc_plane_words(G, W) * sizeof(int); }   // one tile: four planes

size_t acc_smem_bytes(int G, int W, int ncw, int pt, int stages) {
  return (size_t)stages * 7 * acc_chunk(ncw, pt) * sizeof(float) + 2 * acc_tile_bytes(G, W);
}

// A block works through scheduling units u = 0, 1, 2, ... (each a run of consecutive scatterers named by a ticket of the
// global counter).  Unit u + `ahead` is prepared by the warp that is first to enter unit u: its lane 0 draws the ticket with an
// asynchronous atomicAdd, keeps the value in a register while the reduction is in flight and publishes the unit (start,
// end) at the end of its current chunk, long before anybody needs it.  Nobody spins on a lock; readers poll the
// sequence number, all lanes together.
struct PendingUnit {
  unsigned ticket, unit;
  bool pending;
};

struct UnitTable {
  unsigned start0, end0, seq0;   // shared-memory addresses of the three rings
};

__device__ __forceinline__ void publish_unit(const AccParams& p, const UnitTable& ut, PendingUnit& t) {
  if (t.pending) {
    unsigned long long start = 0, end = 0;   // beyond the last ticket: an empty unit = end of work
    if (t.ticket < p.n_big) {                // whole units, visited in a scattered order
      start = (((unsigned long long)t.ticket * p.sc_stride) % p.n_big) * p.superchunk;
      end = start + p.superchunk;
    } else if (t.ticket < p.n_units) {       // the last round: shorter units, in input order
      start = p.tail_start + (unsigned long long)(t.ticket - p.n_big) * p.sc_small;
      end = (start + p.sc_small < p.n) ? start + p.sc_small : p.n;
    }
    const unsigned slot = t.unit & (kRing - 1);
    sh::st64(ut.start0 + 8u * slot, start);
    sh::st64(ut.end0 + 8u * slot, end);
    sh::st_release(ut.seq0 + 4u * slot, (int)(t.unit + 1u));
    t.pending = false;
  }
}

// A stream of chunks through the block's units (one for the copies, one for the reads): the current unit and the run
// of it that is left, in registers.  The unit table is consulted only when a unit is exhausted.
struct ChunkStream {
  unsigned long long base;   // the next chunk starts here
  unsigned left;             // scatterers of the current unit not yet handed out (0: the unit is exhausted)
  unsigned unit;             // index of the next unit to open
  bool stop;                 // the end of work has been seen
};

// Opens unit s.unit (waits for its publication, all lanes together).  An empty unit is the end of work.
__device__ __forceinline__ void stream_open(const UnitTable& ut, ChunkStream& s) {
  const unsigned slot = s.unit & (kRing - 1);
  while ((unsigned)sh::ld_acquire(ut.seq0 + 4u * slot) != s.unit + 1u) __nanosleep(64);
  s.base = sh::ld64(ut.start0 + 8u * slot);
  const unsigned long long end = sh::ld64(ut.end0 + 8u * slot);
  s.left = (unsigned)(end - s.base);   // a unit is shorter than 2^32 scatterers (sim_api.cu)
  s.stop = end == 0ull;
  ++s.unit;
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

// true mod for the (rare) places that need the bin itself: N is any integer >= 1
__device__ __forceinline__ int pmod(int a, int n) {
  const int r = a % n;
  return r < 0 ? r + n : r;
}

// One contribution that left the tile (or never used it): exact-enough fp64 global reductions.
__device__ __forceinline__ void global_add(const AccParams& p, int g0, int k, float w1, float2 c) {
  const int bin = pmod(k, p.N);
  const double w1d = (double)w1, w0d = 1.0 - w1d;
  if (g0 >= 0) {
    double* t = reinterpret_cast<double*>(p.T64 + (size_t)g0 * p.N + bin);
    atomicAdd(t, w0d * (double)c.x);
    atomicAdd(t + 1, w0d * (double)c.y);
  }
  if (g0 + 1 < p.G) {
    double* t = reinterpret_cast<double*>(p.T64 + (size_t)(g0 + 1) * p.N + bin);
    atomicAdd(t, w1d * (double)c.x);
    atomicAdd(t + 1, w1d * (double)c.y);
  }
}

template <int NCW, int PT, int IL, int MODE, bool DBG, bool LUT>
__global__ void __launch_bounds__(NCW * 32, NCW <= 8 ? 2 : 1) acc_kernel(AccParams p) {
  constexpr int CH = NCW * 32 * PT, SL = 32 * PT;
  constexpr unsigned kStageBytes = 7u * CH * 4u;
  constexpr unsigned kFull = 0xffffffffu;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  __shared__ __align__(8) unsigned long long s_ustart[kRing], s_uend[kRing];
  __shared__ int s_useq[kRing];
  __shared__ int s_claimed;             // units that some warp has entered (the first one in prepares unit + 2)
  __shared__ int s_slot[4][kSlotInts];
  // per tile b, one phase per epoch that uses it (NCW arrivals each): "every warp has finished the epoch" and "every warp
  // has drained its share of it".  Waiters sleep in hardware (try_wait with a suspend hint) instead of spinning.
  __shared__ __align__(8) unsigned long long s_bar_complete[2], s_bar_drained[2];
  __shared__ int s_shares[2];           // warps that have drained their share of the completed epoch of tile b

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int S = p.stages, EC = p.epoch_chunks;
  const int G = p.G, W = p.W, RS = p.row_words;
  const unsigned stage0 = sh::addr(smem_raw);
  const unsigned tile0 = stage0 + (unsigned)S * kStageBytes;     // int [2 tiles][4 planes: L.re, L.im, U.re, U.im][G + 1][RS]
  const unsigned plane_bytes = (unsigned)p.plane_words * 4u, tile_bytes = 4u * plane_bytes;
  const UnitTable ut{sh::addr(&s_ustart[0]), sh::addr(&s_uend[0]), sh::addr(&s_useq[0])};
  const unsigned claimed_a = sh::addr(&s_claimed);
  const unsigned complete0 = sh::addr(&s_bar_complete[0]), drained0 = sh::addr(&s_bar_drained[0]);
  const unsigned shares0 = sh::addr(&s_shares[0]);
  const unsigned slot0 = sh::addr(&s_slot[0][0]);
  // the copies run one chunk ahead of the reads: entering unit u, a warp prepares unit u + ahead, which no copy can
  // need before the end of the chunk in which it is published
  const unsigned ahead = 2u;   // (two stages: the copies are one chunk ahead of the reads, at most one unit ahead)
  const unsigned e0 = (unsigned)lane * PT;             // this lane's first scatterer in the warp's slice
  const unsigned slice_lo = (unsigned)warp * SL;       // the warp's slice in a chunk
  const unsigned lane_smem = stage0 + (slice_lo + e0) * 4u;   // this lane's PT scatterers in stage 0, array 0

  for (int i = tid; i < kRing; i += NCW * 32) sh::st(ut.seq0 + 4u * i, 0);
  if (tid < 4) sh::st(slot0 + 4u * kSlotInts * tid + 4 * kSlotState, kSlotUnset);
  if (tid < 2) {
    sh::mbar_init(complete0 + 8u * tid, NCW);
    sh::mbar_init(drained0 + 8u * tid, NCW);
    sh::st(shares0 + 4u * tid, 0);
    sh::mbar_fence_init();
  }
  __syncthreads();
  if (tid == 0) {   // the first `ahead` units are static (tickets b and b + grid of block b): no round trip to the counter
    sh::st(claimed_a, 0);
    for (unsigned u = 0; u < ahead; ++u) {
      PendingUnit t{blockIdx.x + u * gridDim.x, u, true};
      publish_unit(p, ut, t);
    }
  }
  __syncthreads();
  const unsigned ticket0 = ahead * gridDim.x;   // the counter hands out the tickets after the static ones

  PendingUnit tk{0u, 0u, false};
  // This lane's PT scatterers of the next chunk of the copy stream (7 x 16 bytes) -> its place in stage `st`; one commit
  // group per chunk, empty beyond the end of the input.  PT = 2 lanes pair up: the even lane copies for both.
  // One stream of chunks: the chunk copied in an iteration is the one read in the next (two stages).
  ChunkStream cs{0ull, 0u, 0u, false};
  unsigned long long rd_base = 0ull;   // the chunk to read next (copied one iteration ago): first scatterer,
  unsigned rd_nv = 0u;                 // valid count (0: none, the end of work has been reached)
  unsigned long long cp_base = 0ull;   // the chunk copied last
  unsigned cp_nv = 0u;
  bool cp_first = false, rd_first = false;   // the chunk is the first of its scheduling unit
  auto copy_chunk = [&](unsigned st) {
    cp_nv = 0u;
    cp_first = false;
    if (cs.left == 0u && !cs.stop) {   // (rare) the next unit
      stream_open(ut, cs);
      cp_first = true;
      // the first warp to enter a unit (index cs.unit - 1) prepares a later one
      if (!cs.stop) {
        if (lane == 0 && sh::cas(claimed_a, (int)cs.unit - 1, (int)cs.unit) == (int)cs.unit - 1) {
          publish_unit(p, ut, tk);   // (units of a single chunk: this warp's previous ticket may still be pending)
          tk.ticket = atomicAdd(&p.counters[kCtrTicket], 1u) + ticket0;   // in flight until the end of this chunk
          tk.unit = cs.unit - 1u + ahead;
          tk.pending = true;
        }
        __syncwarp();
      }
    }
    if (!cs.stop) {
      const unsigned nv = min(cs.left, (unsigned)CH), n4 = nv & ~3u;
      cs.left -= nv;
      cp_base = cs.base;
      cp_nv = nv;
      const unsigned o4 = (slice_lo + e0) & ~3u;                    // first scatterer of this lane's 16-byte group
      if ((PT == 4 || !(lane & 1)) && o4 + 4u <= n4) {
        const unsigned dst = stage0 + st * kStageBytes + o4 * 4u;
        const unsigned long long g = cs.base + o4;
        sh::cp_async16(dst + 0u * CH * 4u, p.x + g);
        sh::cp_async16(dst + 1u * CH * 4u, p.y + g);
        sh::cp_async16(dst + 2u * CH * 4u, p.z + g);
        sh::cp_async16(dst + 3u * CH * 4u, p.vx + g);
        sh::cp_async16(dst + 4u * CH * 4u, p.vy + g);
        sh::cp_async16(dst + 5u * CH * 4u, p.vz + g);
        sh::cp_async16(dst + 6u * CH * 4u, p.s0dA + g);
      }
      cs.base += CH;
    }
    sh::cp_async_commit();
  };
  if (!DBG) {
    for (unsigned a = 4u * tid; a < 2u * tile_bytes; a += 4u * NCW * 32) sh::st(tile0 + a, 0);
    __syncthreads();
  }
  // Everything up to here touched shared memory only: the launch may have started while the kernel before it in the
  // stream was still running (programmatic dependent launch: the finalize kernel of the previous update signals it
  // early; behind any other kernel the launch is serialised as usual).  Nothing the caller owns and nothing in the
  // workspace is read before this wait: a kernel of the caller's that writes the scatterer arrays earlier in the
  // stream (a surface update) is complete and visible from here on, and so are the accumulator and the ticket counter.
  asm volatile("griddepcontrol.wait;" ::: "memory");
  copy_chunk(0u);   // chunk 0 is in flight (two stages: the copies run one chunk ahead of the reads)
  rd_base = cp_base;
  rd_nv = cp_nv;
  rd_first = cp_first;

  // Step A7: this warp's share (gates [g_lo, g_hi)) of the tile of a completed epoch d -> T64, cells zeroed; the last
  // warp to finish its share hands the tile back.  Gate g = lower halves of row g + 1 (scatterers with g0 = g) + upper
  // halves of row g (g0 = g - 1); row 0 of L and row G of U only collect the halves that fall outside the window: never
  // read, never zeroed.  One lane = two consecutive bins of one gate: four 8-byte loads.
  const int g_lo = (int)(((long long)G * warp) / NCW), g_hi = (int)(((long long)G * (warp + 1)) / NCW);
  const int pairs = RS >> 1;
  auto drain_share = [&](unsigned d) {
    const unsigned b = d & 1u;
    const unsigned slot = slot0 + 4u * kSlotInts * (d & 3u);
    if (sh::ld(slot + 4 * kSlotState) == kSlotReady) {
      const int k0 = pmod(sh::ld(slot + 4 * kSlotK0), p.N), ex = sh::ld(slot + 4 * kSlotEx);
      const double inv_s = __hiloint2double((1023 - ex) << 20, 0);
      const unsigned tile = tile0 + b * tile_bytes;
      const int nitem = (g_hi - g_lo) * pairs;
      // it / pairs = umulhi(it, ceil(2^32 / pairs)): exact while it < 2^32 / pairs (the error of the rounded-up reciprocal,
      // < pairs * 2^-32 per unit of `it`, must stay below one): pairs <= 1026 (window option <= 2048) and nitem <=
      // 129 * 1026 are far inside; pairs >= 2 (a row has at least four words) keeps the reciprocal in 32 bits
      const unsigned inv_pairs = (unsigned)((0x100000000ull + (unsigned long long)pairs - 1ull) / (unsigned long long)pairs);
      for (int it = lane; it < nitem; it += 32) {
        const int gi_ = (int)__umulhi((unsigned)it, inv_pairs);
        const int g = g_lo + gi_, q2 = (it - gi_ * pairs) * 2;
        const unsigned aL = tile + 4u * (unsigned)((g + 1) * RS + q2), aU = tile + 2u * plane_bytes + 4u * (unsigned)(g * RS + q2);
        const int2 lr = sh::ld2(aL), li = sh::ld2(aL + plane_bytes), ur = sh::ld2(aU), ui = sh::ld2(aU + plane_bytes);
        if (lr.x | lr.y | li.x | li.y | ur.x | ur.y | ui.x | ui.y) {
          const int2 z2 = make_int2(0, 0);
          sh::st2(aL, z2);
          sh::st2(aL + plane_bytes, z2);
          sh::st2(aU, z2);
          sh::st2(aU + plane_bytes, z2);
          const int re[2] = {lr.x + ur.x, lr.y + ur.y};
          const int im[2] = {li.x + ui.x, li.y + ui.y};
  #pragma unroll
          for (int c = 0; c < 2; ++c) {
            if (re[c] | im[c]) {   // (columns >= W are never written)
              int bin = k0 + q2 + c;
              bin -= bin >= p.N ? p.N : 0;
              double* t = reinterpret_cast<double*>(p.T64 + (size_t)g * p.N + bin);
              atomicAdd(t, (double)re[c] * inv_s);
              atomicAdd(t + 1, (double)im[c] * inv_s);
            }
          }
        }
      }
    }
    __syncwarp();
    if (lane == 0) {
      if (sh::atom_add_acq_rel(shares0 + 4u * b, 1) == NCW - 1) {   // every share is out: the slot goes back ...
        sh::st(shares0 + 4u * b, 0);
        sh::st(slot + 4 * kSlotState, kSlotUnset);
      }
      sh::mbar_arrive(drained0 + 8u * b);                             // ... and, with the last arrival, the tile
    }
    __syncwarp();
  };
  // Drains the shares of the epochs before `upto` that are complete; called at chunk boundaries (cheap when nothing is
  // pending).  block = true: waits for the completion (end of the kernel, or a tile that this warp needs back).
  unsigned dpend = 0;   // the oldest epoch whose share this warp has not drained yet
  auto try_drain = [&](unsigned upto, bool block) {
    while (dpend < upto) {
      const unsigned b = dpend & 1u;
      const unsigned par = (dpend >> 1) & 1u;
      if (block) sh::mbar_wait_sleepy(complete0 + 8u * b, par, 2000u);   // a warp that is ahead sleeps: no issue slots taken
      else if (!sh::mbar_test(complete0 + 8u * b, par)) return;
      drain_share(dpend);
      ++dpend;
    }
  };

  // lane-dependent issue order of a scatterer's four reductions: bit 0 swaps re/im, bit 1 swaps lower/upper
  const bool sw_ri = lane & 1, sw_lu = (lane >> 1) & 1;
  unsigned off_b0 = (sw_lu ? 2u : 0u) * plane_bytes + (sw_ri ? plane_bytes : 0u);   // plane of (value a0, weight wB)
  int d_ri = sw_ri ? -(int)plane_bytes : (int)plane_bytes;                          // a0 -> a1
  int d_lu = sw_lu ? -2 * (int)plane_bytes : 2 * (int)plane_bytes;                  // wB -> wA
  const int RS4 = 4 * RS;
  off_b0 += (unsigned)RS4;   // the +1 row offset of the padded tile folded in
  // opaque to the compiler: kept in three registers instead of being re-derived from the lane number for every group of
  // scatterers (14 instructions per scatterer in the profile of the version without this line)
  asm volatile("" : "+r"(off_b0), "+r"(d_ri), "+r"(d_lu));
  unsigned stg = 0;
  unsigned escapes = 0, fallbacks = 0;
  bool more = true;
  const unsigned fx_span = (unsigned)(p.fx_cap - 11) << 23;   // admitted |c| s: [2^11, 2^fx_cap]

  for (unsigned e = 0; more; ++e) {
    const unsigned slot = slot0 + 4u * kSlotInts * (e & 3u);
    // The index export has no tiles and hence no tile hand-over to keep the warps of a block within two epochs of each
    // other; without a bound a warp could run more than kRing units ahead of a sibling and overwrite unit-table entries
    // the sibling has not read.  Every warp walks the same chunks and epochs (the stream is block-uniform), so a
    // barrier per epoch is safe, and cheap enough for a debug path.
    if (DBG) __syncthreads();
    if (!DBG && e >= 2) {   // the tile of epoch e-2 must be back: this warp's own share first, then everybody else's
      try_drain(e - 1u, true);
      sh::mbar_wait_sleepy(drained0 + 8u * (e & 1u), ((e >> 1) - 1u) & 1u, 2000u);
    }
    // tile base of this lane's first reduction, the +1 row offset of the padded tile folded in
    unsigned tile_b = tile0 + (e & 1u) * tile_bytes + off_b0;
    asm volatile("" : "+r"(tile_b));
    const unsigned dump_b = tile_b + (unsigned)(G * RS4 + 4 * lane);   // row G + 1 onwards of this lane's first plane
    bool have = false;         // this warp holds the epoch's parameters
    int k0 = 0, lo_bits = 0;
    float s = 0.0f, sS = 0.0f, sO = 0.0f;
    int ci = 0;
    for (; ci < EC; ++ci) {
      if (!DBG && dpend < e && sh::mbar_test(complete0 + 8u * (dpend & 1u), (dpend >> 1) & 1u)) try_drain(e, false);
      // a scheduling unit that is not whole epochs (the ragged end of the input) ends its epoch early: the next unit lies
      // elsewhere in the scene and gets its own Doppler window
      if (ci > 0 && rd_first) break;
      // the next chunk goes into the stage that was read one iteration ago; then this lane's copies of the chunk to read
      // (one group older) must have landed
      copy_chunk(stg ^ 1u);
      sh::cp_async_wait<1>();
      if (PT == 2) __syncwarp();   // the even lane's copy serves its odd neighbour
      if (rd_nv == 0u) {           // block-uniform: end of work
        more = false;
        break;
      }
      const unsigned long long base = rd_base;
      const unsigned nvalid = rd_nv;
      rd_base = cp_base;
      rd_nv = cp_nv;
      rd_first = cp_first;

      // ---- step A1: this lane's PT scatterers, shared-memory stage -> registers; the slice is refilled at once ----
      Vec<PT> x, y, z, vx, vy, vz, s0;
      const unsigned off = slice_lo + e0;         // offset in the chunk
      if (off + PT <= (nvalid & ~3u)) {
        const unsigned a = lane_smem + stg * kStageBytes;
        x.load(a + 0u * CH * 4u);
        y.load(a + 1u * CH * 4u);
        z.load(a + 2u * CH * 4u);
        vx.load(a + 3u * CH * 4u);
        vy.load(a + 4u * CH * 4u);
        vz.load(a + 5u * CH * 4u);
        s0.load(a + 6u * CH * 4u);
      } else {  // ragged end of the input: not covered by the 16-byte bulk copies; s0dA = 0 contributes nothing
#pragma unroll
        for (int j = 0; j < PT; ++j) {
          const bool v = off + j < nvalid;
          const unsigned long long i = base + off + j;
          x.v[j] = v ? p.x[i] : 0.0f;
          y.v[j] = v ? p.y[i] : 0.0f;
          z.v[j] = v ? p.z[i] : 0.0f;
          vx.v[j] = v ? p.vx[i] : 0.0f;
          vy.v[j] = v ? p.vy[i] : 0.0f;
          vz.v[j] = v ? p.vz[i] : 0.0f;
          s0.v[j] = v ? p.s0dA[i] : 0.0f;
        }
      }
      stg ^= 1u;

#pragma unroll
      for (int gi = 0; gi < PT; gi += IL) {   // IL scatterers in flight per lane at a time
        // ---- steps A2-A5 ----
        bool ok[IL];
        Pre q[IL];
        Fx fx[IL];
        float2 c[IL];
        int ab[IL];
        bool any = false;
  #pragma unroll
        for (int j = 0; j < IL; ++j) {
          ok[j] = DBG ? (off + gi + j < nvalid) : (s0.v[gi + j] > 0.0f);   // s0dA <= 0 or NaN: dead (not consulted by the index export)
          q[j] = pre_part<MODE>(p, x.v[gi + j], y.v[gi + j], z.v[gi + j], ok[j]);
          any |= ok[j];
        }
        if (!__any_sync(kFull, any)) {   // warp-uniform: the whole warp is dark
          if (DBG) {
  #pragma unroll
            for (int j = 0; j < IL; ++j)
              if (off + gi + j < nvalid) {
                p.dbg_g0[base + off + gi + j] = SIM_GATE_NONE;
                p.dbg_k[base + off + gi + j] = -1;
              }
          }
          continue;
        }
        Idx cx[IL];   // canonical mode only
        if (MODE == kIdxCanonical) {
  #pragma unroll
          for (int j = 0; j < IL; ++j) {
            ok[j] = ok[j] && canonical(p, q[j].dx, q[j].dy, q[j].dz, vx.v[gi + j], vy.v[gi + j], vz.v[gi + j], cx[j]);
            // g0 and a 20-bit weight for the tile path; the bin itself (no fraction bits)
            fx[j].gfx = (cx[j].g0 << kFracBits) + min((int)(cx[j].w1 * (float)kFxOne), kFxOne - 1);
            fx[j].kfx = cx[j].k;
            fx[j].fr = cx[j].fr * 4294967296.0f;   // cycles -> units of 2^-32 cycles
          }
        } else {
          // polynomial path straight through for all IL scatterers; the guard-band cases are re-decided in the cold block
  #pragma unroll
          for (int j = 0; j < IL; ++j)
            fx[j] = index_fx<MODE>(p, q[j], x.v[gi + j], y.v[gi + j], z.v[gi + j], vx.v[gi + j], vy.v[gi + j], vz.v[gi + j]);
        }
        if (!DBG) {
          if (LUT) {
  #pragma unroll
            for (int j = 0; j < IL; ++j) {
              float A;
              c[j] = amplitude_t<true>(p, x.v[gi + j], y.v[gi + j], z.v[gi + j], (float)fx[j].gfx, fx[j].fr * kFrUnit, s0.v[gi + j], A);
              ab[j] = __float_as_int(A);
              ok[j] = ok[j] && A > 0.0f;   // outside the recorded antenna pattern: contributes nothing
            }
          } else {   // two scatterers per packed fp32 instruction
  #pragma unroll
            for (int j = 0; j < IL; j += 2) {
              float2 A, cre, cim;
              amplitude_pair(p, make_float2(x.v[gi + j], x.v[gi + j + 1]), make_float2(y.v[gi + j], y.v[gi + j + 1]),
                             make_float2(z.v[gi + j], z.v[gi + j + 1]), make_float2((float)fx[j].gfx, (float)fx[j + 1].gfx),
                             make_float2(fx[j].fr, fx[j + 1].fr), make_float2(s0.v[gi + j], s0.v[gi + j + 1]), A, cre, cim);
              c[j] = make_float2(cre.x, cim.x);
              c[j + 1] = make_float2(cre.y, cim.y);
              ab[j] = __float_as_int(A.x);
              ab[j + 1] = __float_as_int(A.y);
            }
          }
        }
        // ---- gate, bin, weight and the guard-band test, from the two fixed-point coordinates ----
        int g0[IL], k[IL];
        bool near[IL];
        any = false;
  #pragma unroll
        for (int j = 0; j < IL; ++j) {
          g0[j] = fx[j].gfx >> kFracBits;
          if (MODE == kIdxCanonical) {
            k[j] = fx[j].kfx;
            near[j] = false;
          } else {
            k[j] = fx_bin<MODE>(p, fx[j]);
            near[j] = ok[j] && fx_near<MODE>(p, fx[j]);
          }
          any |= ok[j];
        }
        if (DBG) {
          bool any_near = false;
  #pragma unroll
          for (int j = 0; j < IL; ++j) any_near |= near[j];
          if (__any_sync(kFull, any_near)) {
  #pragma unroll
            for (int j = 0; j < IL; ++j) {
              if (near[j]) {
                ++fallbacks;
                Idx t;
                ok[j] = canonical(p, __dsub_rn((double)x.v[gi + j], p.sx), __dsub_rn((double)y.v[gi + j], p.sy),
                                  __dsub_rn((double)z.v[gi + j], p.sz), vx.v[gi + j], vy.v[gi + j], vz.v[gi + j], t);
                g0[j] = t.g0;
                k[j] = t.k;
              }
            }
          }
  #pragma unroll
          for (int j = 0; j < IL; ++j)
            if (off + gi + j < nvalid) {
              p.dbg_g0[base + off + gi + j] = ok[j] ? g0[j] : SIM_GATE_NONE;
              p.dbg_k[base + off + gi + j] = ok[j] ? pmod(k[j], p.N) : -1;
            }
          continue;
        }
        const unsigned okm = __ballot_sync(kFull, any);
        if (okm == 0) continue;

        // ---- epoch parameters: the first warp with something to add decides them ----
        if (!have) {
          int st = 0;
          if (lane == 0) {
            st = sh::ld_acquire(slot + 4 * kSlotState);
            if (st != kSlotReady) st = sh::cas(slot + 4 * kSlotState, kSlotUnset, kSlotClaimed);
          }
          st = __shfl_sync(kFull, st, 0);
          if (st == kSlotUnset) {  // this warp won the claim: window and scale from its own scatterers
            int kk = 0;
  #pragma unroll
            for (int j = IL - 1; j >= 0; --j) kk = ok[j] ? k[j] : kk;
            const int kref = __shfl_sync(kFull, kk, __ffs(okm) - 1);
            int dmin = INT_MAX, dmax = INT_MIN, cnt = 0, slog = 0;
  #pragma unroll
            for (int j = 0; j < IL; ++j) {
              const int d = k[j] - kref;                                     // bins are unwrapped here: plain offsets
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
              const int centre = ((long long)dmax - dmin < W) ? kref + ((dmin + dmax + 1) >> 1) : kref;
              const int E = (slog / cnt) >> 7;                      // biased exponent of the geometric mean
              const int ex = max(-100, min(120, p.fx_target - (E - 127)));   // gmean * 2^ex in [2^16, 2^17) (default)
              sh::st(slot + 4 * kSlotK0, centre - (W >> 1));
              sh::st(slot + 4 * kSlotEx, ex);
              sh::st_release(slot + 4 * kSlotState, kSlotReady);
            }
            __syncwarp();
          } else if (st == kSlotClaimed) {
            while (sh::ld_acquire(slot + 4 * kSlotState) != kSlotReady) __nanosleep(64);
          }
          k0 = sh::ld(slot + 4 * kSlotK0);
          const int ex = sh::ld(slot + 4 * kSlotEx);
          s = __int_as_float((ex + 127) << 23);
          sS = (sw_lu ? -s : s) * p.w_scale;
          sO = sw_lu ? s : 0.0f;
          lo_bits = (11 - ex + 127) << 23;                    // bits of 2^11 / s
          have = true;
        }

        // ---- step A6: native int32 shared-memory reductions; whatever does not fit takes the cold block ----
        bool slow_any = false;
        bool slow[IL];
        int r0[IL], r1[IL], r2[IL], r3[IL];   // round(value * weight * s) of the four reductions (1.5 * 2^23 trick), pairwise
  #pragma unroll
        for (int j = 0; j < IL; j += 2) {
          const float2 fw = make_float2((float)(fx[j].gfx & (kFxOne - 1)), (float)(fx[j + 1].gfx & (kFxOne - 1)));
          const float2 wAs = fma2(fw, bc(sS), bc(sO)), wBs = fma2(wAs, bc(-1.0f), bc(s));   // (w1, w0) s, or (w0, w1) s on swapped lanes
          const float2 a0 = make_float2(sw_ri ? c[j].y : c[j].x, sw_ri ? c[j + 1].y : c[j + 1].x);
          const float2 a1 = make_float2(sw_ri ? c[j].x : c[j].y, sw_ri ? c[j + 1].x : c[j + 1].y);
          const float2 v0 = fma2(a0, wBs, bc(12582912.0f)), v1 = fma2(a1, wBs, bc(12582912.0f));
          const float2 v2 = fma2(a0, wAs, bc(12582912.0f)), v3 = fma2(a1, wAs, bc(12582912.0f));
          r0[j] = __float_as_int(v0.x) - 0x4B400000; r0[j + 1] = __float_as_int(v0.y) - 0x4B400000;
          r1[j] = __float_as_int(v1.x) - 0x4B400000; r1[j + 1] = __float_as_int(v1.y) - 0x4B400000;
          r2[j] = __float_as_int(v2.x) - 0x4B400000; r2[j + 1] = __float_as_int(v2.y) - 0x4B400000;
          r3[j] = __float_as_int(v3.x) - 0x4B400000; r3[j + 1] = __float_as_int(v3.y) - 0x4B400000;
        }
  #pragma unroll
        for (int j = 0; j < IL; ++j) {
          const int kw = k[j] - k0;
          const bool fits = ok[j] && !near[j] && (unsigned)kw < (unsigned)W && (unsigned)(ab[j] - lo_bits) <= fx_span;
          const unsigned adr = fits ? tile_b + (unsigned)(g0[j] * RS4 + 4 * kw) : dump_b;   // (tile cell, or this lane's dump word)
          sh::red_add(adr, r0[j]);
          sh::red_add(adr + d_ri, r1[j]);
          sh::red_add(adr + d_lu, r2[j]);
          sh::red_add(adr + d_lu + d_ri, r3[j]);
          slow[j] = ok[j] && !fits;
          slow_any |= slow[j];
        }
        if (__any_sync(kFull, slow_any)) {  // rare: guard band (canonical sequence decides), window or range escape
  #pragma unroll
          for (int j = 0; j < IL; ++j) {
            if (slow[j]) {
              Idx t;
              if (MODE == kIdxCanonical) {
                t = cx[j];
              } else if (!near[j]) {
                // outside the Doppler window or the fixed-point range of the epoch: the polynomial path's gate, bin,
                // weight and amplitude stand, only the tile cannot take them
                global_add(p, g0[j], k[j], (float)(fx[j].gfx & (kFxOne - 1)) * p.w_scale, c[j]);
                ++escapes;
                continue;
              } else {
                ++fallbacks;
                // the canonical sequence for every scatterer that leaves the tile (guard band or not: it is exact);
                // offsets recomputed here (three subtractions) rather than kept alive across the amplitude for this rare case
                const bool okj = canonical(p, __dsub_rn((double)x.v[gi + j], p.sx), __dsub_rn((double)y.v[gi + j], p.sy),
                                           __dsub_rn((double)z.v[gi + j], p.sz), vx.v[gi + j], vy.v[gi + j], vz.v[gi + j], t);
                if (!okj) continue;
                float A;
                c[j] = amplitude_t<LUT>(p, x.v[gi + j], y.v[gi + j], z.v[gi + j], t.gfx, t.fr, s0.v[gi + j], A);
                if (!(A > 0.0f)) continue;
              }
              global_add(p, t.g0, t.k, t.w1, c[j]);
              ++escapes;
            }
          }
        }
      }
      // the ticket drawn when this warp was first into a unit (at the top of this chunk) has had the whole chunk to come
      // back: the unit is published before this warp can wait for anybody
      if (lane == 0) publish_unit(p, ut, tk);
      __syncwarp();
    }

    // ---- end of an epoch (or of the input inside one): the last warp out declares the tile complete ----
    if (!DBG) {
      __syncwarp();
      if (lane == 0) sh::mbar_arrive(complete0 + 8u * (e & 1u));   // the last warp out completes the phase: the tile can be drained
      __syncwarp();
      if (!more) try_drain(e + 1u, true);   // the end of the input: the shares of the last epochs
    }
  }
  if (lane == 0) publish_unit(p, ut, tk);
  if (escapes) atomicAdd(&p.counters[kCtrEscape], escapes);
  if (fallbacks) atomicAdd(&p.counters[kCtrFallback], fallbacks);
  // the last block out leaves the scheduling counter at zero for the next launch (every block has drawn its last ticket
  // before it gets here): no memset between launches
  __syncthreads();
  if (tid == 0 && atomicAdd(&p.counters[kCtrDone], 1u) == gridDim.x - 1u) {
    p.counters[kCtrDone] = 0u;
    p.counters[kCtrTicket] = 0u;
  }
}

// ---------------------------------------------------------------------------------------------
// Variant 0: reference kernel.  One scatterer per thread, the canonical sequence for every scatterer, fp64 global
// reductions.  Plain on purpose: it is the A/B partner of the production kernel.
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) acc_reference_kernel(AccParams p) {
  const unsigned long long stride = (unsigned long long)gridDim.x * blockDim.x;
  for (unsigned long long i = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; i < p.n; i += stride) {
    const float s0 = p.s0dA[i];
    if (!(s0 > 0.0f)) continue;
    const float xf = p.x[i], yf = p.y[i], zf = p.z[i];
    Idx ix;
    if (!canonical(p, __dsub_rn((double)xf, p.sx), __dsub_rn((double)yf, p.sy), __dsub_rn((double)zf, p.sz), p.vx[i], p.vy[i],
                   p.vz[i], ix))
      continue;
    float A;
    const float2 c = amplitude(p, xf, yf, zf, ix.gfx, ix.fr, s0, A);
    global_add(p, ix.g0, ix.k, ix.w1, c);
  }
}

// T64 -> spectrum slot (complex64), T64 re-zeroed.  add != 0: the slot already holds earlier batches of this update
// (SIM_ACC_APPEND).
__global__ void __launch_bounds__(256) acc_finalize_kernel(double2* __restrict__ T64, float2* __restrict__ T, int cells, int add) {
  // the next accumulation launch may start now: it sets up its shared memory, then waits for this grid to complete
  // before it reads anything from global memory (programmatic dependent launch; see acc_kernel)
  asm volatile("griddepcontrol.launch_dependents;");
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= cells) return;
  const double2 v = T64[i];
  float2 o = make_float2((float)v.x, (float)v.y);
  if (add) {
    const float2 t = T[i];
    o.x += t.x;
    o.y += t.y;
  }
  T[i] = o;
  if (v.x != 0.0 || v.y != 0.0) T64[i] = make_double2(0.0, 0.0);
}

cudaError_t launch_finalize(double2* T64, float2* T, int cells, bool add, cudaStream_t st, int* launches) {
  acc_finalize_kernel<<<(cells + 255) / 256, 256, 0, st>>>(T64, T, cells, add ? 1 : 0);
  ++*launches;
  return cudaGetLastError();
}

// Which index routine a launch uses: the polynomial path of the configured Doppler source when the host found
// its error bounds covered by the guard band, else the canonical sequence everywhere.
int acc_index_mode(const AccParams& p) {
  if (!p.index_path) return kIdxCanonical;
  if (p.doppler_mode == SIM_DOPPLER_PULSE_PAIR) return p.pp_ok ? kIdxFastPulsePair : kIdxCanonical;
  return p.fast_ok ? kIdxFast : kIdxCanonical;
}

// ---------------------------------------------------------------------------------------------
// Launchers
// ---------------------------------------------------------------------------------------------
typedef void (*AccKernel)(AccParams);

// kind: 0 accumulate with the analytic gain, 1 accumulate with the tabulated gain, 2 index export
static AccKernel acc_kernel_ptr(int ncw, int pt, int il, int mode, int kind) {
#define ACC_MODE(NCW_, PT_, IL_, DBG_, LUT_)                                                                   \
  (mode == kIdxFast ? acc_kernel<NCW_, PT_, IL_, kIdxFast, DBG_, LUT_>                                         \
   : mode == kIdxFastPulsePair ? acc_kernel<NCW_, PT_, IL_, kIdxFastPulsePair, DBG_, LUT_>                     \
                               : acc_kernel<NCW_, PT_, IL_, kIdxCanonical, DBG_, LUT_>)
#define ACC_CASE(NCW_, PT_, IL_)                                                                               \
  if (ncw == NCW_ && pt == PT_ && il == IL_)                                                                   \
    return kind == 2 ? ACC_MODE(NCW_, PT_, IL_, true, false) : kind == 1 ? ACC_MODE(NCW_, PT_, IL_, false, true) \
                                                                         : ACC_MODE(NCW_, PT_, IL_, false, false);
  ACC_CASE(8, 4, 4) ACC_CASE(8, 4, 2) ACC_CASE(8, 2, 2) ACC_CASE(16, 4, 4)
#undef ACC_CASE
#undef ACC_MODE
  return nullptr;
}

bool acc_supported(int ncw, int pt, int il) { return acc_kernel_ptr(ncw, pt, il, kIdxFast, 0) != nullptr; }

cudaError_t acc_blocks_per_sm(int G, int W, int ncw, int pt, int il, int stages, int* blocks) {
  const size_t smem = acc_smem_bytes(G, W, ncw, pt, stages);
  *blocks = 1 << 30;
  for (int mk = 0; mk < 6; ++mk) {
    const int mode = mk % 3;
    AccKernel k = acc_kernel_ptr(ncw, pt, il, mode, mk / 3);
    if (!k) return cudaErrorInvalidValue;
    cudaError_t e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    int b = 0;
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&b, k, ncw * 32, smem);
    if (e != cudaSuccess) return e;
    if (b < *blocks) *blocks = b;
  }
  return cudaSuccess;
}

// dbg: the same kernel writes (g0, k) per scatterer into p.dbg_g0 / p.dbg_k instead of accumulating.
cudaError_t launch_accumulate(const AccParams& p, int ncw, int pt, int il, int blocks, bool dbg, cudaStream_t st, int* launches) {
  if (p.n == 0) return cudaSuccess;
  const int mode = acc_index_mode(p);
  AccKernel k = acc_kernel_ptr(ncw, pt, il, mode, dbg ? 2 : (p.lut != nullptr ? 1 : 0));
  if (!k) return cudaErrorInvalidValue;
  const size_t smem = acc_smem_bytes(p.G, p.W, ncw, pt, p.stages);
  // per launch: the limit is per function and per device, another handle may have set it for a smaller shape
  cudaError_t e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return e;
  const int grid = (int)(p.n_units < (unsigned)blocks ? p.n_units : (unsigned)blocks);
  cudaLaunchConfig_t cfg{};
  cfg.gridDim = dim3(grid);
  cfg.blockDim = dim3(ncw * 32);
  cfg.dynamicSmemBytes = smem;
  cfg.stream = st;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  // programmatic dependent launch: when the kernel before this one in the stream is the finalize kernel of the previous
  // update (the only one of ours that signals it), this grid may start while that one runs; it waits for it before it
  // reads or writes any global memory (griddepcontrol.wait in acc_kernel), so stream order holds for the caller's
  // arrays too, whatever kernel of the caller's comes before this one.
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  e = cudaLaunchKernelEx(&cfg, k, p);
  ++*launches;
  return e;
}

cudaError_t launch_reference(const AccParams& p, int sm_count, cudaStream_t st, int* launches) {
  if (p.n == 0) return cudaSuccess;
  const unsigned long long want = (p.n + 255) / 256;
  const unsigned long long cap = (unsigned long long)sm_count * 16;
  acc_reference_kernel<<<(int)(want < cap ? want : cap), 256, 0, st>>>(p);
  ++*launches;
  return cudaGetLastError();
}

}  // namespace simk
