// Internal declarations of libsim.so (not part of the ABI; see include/sim.h).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "sim.h"

namespace simk {

constexpr int kAccThreads = 512;              // threads per block of the accumulation kernels
constexpr int kAccPerThread = 4;              // scatterers per thread per chunk (one 128-bit load per array)
constexpr int kAccChunk = kAccThreads * kAccPerThread;
constexpr int kNumCounters = 64;

enum Counter : int {
  kCtrTicket = 0,   // super-chunk ticket of the running accumulation launch
  kCtrMiss = 1,     // contributions that fell outside the shared-memory window (global atomics)
  kCtrFlush = 2,    // tile flushes
};

// Everything the accumulation kernels need, passed by value.
struct AccParams {
  const float *x, *y, *z, *vx, *vy, *vz, *s0dA;
  unsigned long long n;
  double sx, sy, sz;      // satellite position
  double svx, svy, svz;   // satellite velocity
  double rg0;             // range of the centre of gate 0
  double inv_dR;          // 1.0 / gate_spacing
  double two_over_lambda; // 2.0 / wavelength
  double cD;              // (-2.0 * N) / (wavelength * PRF)
  float bx, by, bz;       // unit boresight
  float alpha;            // antenna_alpha
  int G, N;
  float2* T;              // spectrum of the current update, [G][N]
  unsigned int* counters; // kNumCounters device words
  unsigned long long superchunk; // scatterers per scheduling unit (multiple of kAccChunk)
  int W;                  // window bins in shared memory (power of two, <= N)
  int R;                  // replicas (power of two)
  int index_path;         // 0 canonical everywhere, 1 fast path + guard band
};

struct SynParams {
  const float2* ring;     // spectra ring base
  size_t slot_stride;     // float2 elements per slot
  int cap;                // ring capacity
  const float2* tw;       // twiddles exp(+2 pi i j / N), j < N/2
  float2* iq;             // output [n_pulses][G]
  long long x0;           // first pulse of this call
  long long n_pulses;
  long long seg0;         // first segment touched
  long long n_spectra;    // spectra accumulated so far (successor of s exists iff s+1 < n_spectra)
  int G, N, logN, P;
  int GT;                 // gates per block
  int weight_mode;
};

cudaError_t launch_accumulate(const AccParams& p, int variant, int blocks, cudaStream_t st,
                              int* launches);
cudaError_t launch_indices(const AccParams& p, int32_t* g0, int32_t* k, cudaStream_t st,
                           int* launches);
cudaError_t acc_tile_smem_bytes(int G, int W, int R, size_t* bytes);
cudaError_t launch_twiddles(float2* tw, int N, cudaStream_t st, int* launches);
cudaError_t launch_synthesize(const SynParams& p, int n_segments, cudaStream_t st, int* launches);
int synth_gate_tile(int N);

}  // namespace simk
