// Internal declarations of libsim.so (not part of the ABI; see include/sim.h).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "sim.h"

namespace simk {

constexpr int kNumCounters = 64;
constexpr int kSynMaxPass = 12;                // passes of the mixed-radix inverse FFT (N <= 4096 needs at most 7: 3^7, 4 * 3^6, 5 * 3^6)
constexpr int kFracBits = 20;                 // fixed-point fraction bits of the gate / Doppler coordinates

enum Counter : int {
  kCtrTicket = 0,   // scheduling ticket of the running accumulation launch
  kCtrEscape = 1,   // contributions sent to global reductions (guard band, outside the window or the fixed-point range)
  kCtrDone = 2,     // blocks of the running accumulation launch that have finished (the last one out resets the ticket)
  kCtrFallback = 3, // scatterers whose indices were decided by the canonical sequence (guard band)
};

// Everything the accumulation kernels need, passed by value.
struct AccParams {
  const float *x, *y, *z, *vx, *vy, *vz, *s0dA;
  unsigned long long n;
  // ---- canonical fp64 sequence ----
  double sx, sy, sz;      // satellite position
  double svx, svy, svz;   // satellite velocity
  double rg0;             // range of the centre of gate 0
  double inv_dR;          // 1.0 / gate_spacing
  double two_over_lambda; // 2.0 / wavelength
  double cD;              // (-2.0 * N) / (wavelength * PRF)
  double pri, cP;         // pulse-pair Doppler: 1.0 / PRF and (-2.0 * N) / wavelength
  int doppler_mode;       // SIM_DOPPLER_*
  double fr0;             // frac(rg0 * 2 / lambda), exact to ~1e-17
  double fr0m;            // fr0 + 1.5 * 2^28 (the magic number of the phase read rides in the addend)
  // ---- polynomial index path in u = R^2 - rg0^2: no sqrt, no divide ----
  int index_path;         // 0 canonical everywhere, 1 polynomial path + guard band
  int guard;              // guard band in units of 2^-kFracBits around integer gate boundaries
  int guard_k;            // the same for the Doppler coordinate (wider for the pulse-pair path)
  int fast_ok;            // host-side validity of the polynomial path for this geometry (analytic Doppler)
  int pp_ok;              // ... of the pulse-pair polynomial path
  double neg_rg0sq;       // -(rg0 * rg0), rounded once
  double uw_lo, uw_hi;    // u outside [uw_lo, uw_hi]: outside the gate window by more than half a guard band
  double g1, g2, g3;      // gf = u (g1 + u (g2 + u g3))            = (R - rg0) / dR
  double j0, j1, j2;      // kf = num (j0 + u (j1 + u j2))          = num cD / R
  double cq;              // dR * 2 / lambda: cycles of phase per gate
  double inv_2rg0, two_dR, cP_2rg0;   // pulse-pair polynomial path: 1 / (2 rg0), 2 * gate_spacing, cP / (2 rg0)
  // ---- fp32 amplitude path ----
  float sxh, syh, szh, szl;            // satellite position as float (z as hi + lo)
  float neg_alpha_log2e;               // -antenna_alpha * log2(e)
  float e1x, e1y, e1z, e2x, e2y, e2z;  // orthonormal basis of the plane normal to the boresight
  float e1c, e2c;                      // -r_sat.e1, -r_sat.e2 (with the fp32 basis vectors): d.e1 = r_p.e1 + e1c
  float a0, a1, a2;       // 1/R^2 = a0 + gfx (a1 + gfx a2), gfx = gf * 2^kFracBits
  float w_scale;          // 2^-kFracBits
  // ---- tabulated antenna gain on a u-v grid (reading R9); lut == nullptr: analytic gain ----
  const float2* lut;      // [lut_nv][lut_nu] complex gain, u fastest
  int lut_nu, lut_nv;
  float lut_u0, lut_v0, lut_inv_du, lut_inv_dv;
  int G, N;
  float2* T;              // spectrum slot of the current update, [G][N] (written by the finalize kernel)
  double2* T64;           // fp64 accumulator [G][N]: zero between updates, rounded to T by the finalize kernel
  int32_t *dbg_g0, *dbg_k;   // index export of the production kernel (sim_debug_indices)
  unsigned int* counters; // kNumCounters device words
  unsigned long long superchunk; // scatterers per scheduling unit (whole fixed-point epochs)
  // tickets < n_big: whole units of `superchunk` in the scattered order; then the rest of the input, [tail_start, n), in
  // shorter units of `sc_small` in input order (the last round: blocks finish closer together); n_units in all
  unsigned n_big, n_units;
  unsigned long long tail_start, sc_small;
  int W;                  // Doppler bins of the shared-memory window
  int row_words, plane_words;   // production kernel: tile layout (accumulate.cu)
  int stages, epoch_chunks;  // stages of the copy ring (2); chunks per fixed-point epoch
  int fx_cap, fx_target;     // block floating point: |c| s <= 2^fx_cap admitted; gmean(|c|) s in [2^fx_target, 2^(fx_target+1))
  unsigned long long sc_stride;  // scheduling unit visited by ticket t is (t * sc_stride) mod n_units (coprime)
};

struct SynParams {
  const float2* ring;     // spectra ring base
  size_t slot_stride;     // float2 elements per slot
  int cap;                // ring capacity
  const float2* tw;       // twiddles exp(+2 pi i j / N), j < N
  float2* iq;             // output [n_pulses][G]
  long long x0;           // first pulse of this call
  long long n_pulses;
  long long seg0;         // first segment touched
  long long n_segments;   // segments touched by this call
  long long n_spectra;    // spectra accumulated so far (successor of s exists iff s+1 < n_spectra)
  int G, N, P;
  int GT;                 // gates per block
  int seg_per_block;      // consecutive segments per block (each spectrum is transformed once per run)
  int n_pass, radix[kSynMaxPass];   // Stockham passes: N = product of the radices (4, 2, 3, 5)
  int pass_m[kSynMaxPass], pass_ns[kSynMaxPass], pass_tstep[kSynMaxPass];   // butterflies per signal, product of the earlier radices, twiddle step
  int weight_mode;
};

// production kernel (accumulate.cu): ncw warps per block, pt scatterers per lane per chunk, il in flight per lane
int acc_chunk(int ncw, int pt);
int acc_row_stride(int W);
int acc_plane_words(int G, int W);
size_t acc_smem_bytes(int G, int W, int ncw, int pt, int stages);
bool acc_supported(int ncw, int pt, int il);
cudaError_t acc_blocks_per_sm(int G, int W, int ncw, int pt, int il, int stages, int* blocks);
cudaError_t launch_accumulate(const AccParams& p, int ncw, int pt, int il, int blocks, bool dbg, cudaStream_t st, int* launches);
cudaError_t launch_reference(const AccParams& p, int sm_count, cudaStream_t st, int* launches);
cudaError_t launch_finalize(double2* T64, float2* T, int cells, bool add, cudaStream_t st, int* launches);
// regular mode (regular.cu): Y[n_pulses][G] += per-pulse coherent sums; cudaErrorInvalidConfiguration when G is too
// large for one pulse row per thread in shared memory
cudaError_t launch_regular(const AccParams& a, float2* Y, long long j0, int n_pulses, double prf, int sm_count,
                           size_t smem_optin, cudaStream_t st, int* launches);
// Delay-Doppler burst step (burst.cu): Z[b][k][g] = forward FFT over the 2^logB pulses of burst b, per gate
cudaError_t launch_burst_fft(const float2* Y, float2* Z, long long n_bursts, int logB, int G, cudaStream_t st,
                             int* launches);
cudaError_t launch_twiddles(float2* tw, int N, cudaStream_t st, int* launches);
cudaError_t launch_synthesize(const SynParams& p, cudaStream_t st, int* launches);
void synth_plan(int N, int G, int P, long long n_segments, int sm_count, int* gt, int* seg_per_block);
bool synth_factor(int N, int* radix, int* n_pass);
cudaError_t synth_prepare(int N, int P);

}  // namespace simk
