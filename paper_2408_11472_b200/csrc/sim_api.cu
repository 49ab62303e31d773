// Host side of libsim.so: the C ABI of include/sim.h.  Validation, ring bookkeeping, constant
// derivation in fp64, kernel launches.  No device allocation happens here: everything lives in the
// caller's workspace.
#include <cmath>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <new>
#include <string>

#include "sim_internal.h"

using namespace simk;

namespace {

thread_local std::string g_create_error;

inline size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

struct Layout {
  size_t ring_off, slot_bytes, t64_off, t64_bytes, tw_off, ctr_off, stage_off, stage_buf_bytes, iq_off, iq_bytes, total;
};

Layout make_layout(const sim_config& c) {
  Layout L{};
  size_t off = 0;
  L.ring_off = off;
  L.slot_bytes = align_up((size_t)c.n_gates * c.n_doppler * sizeof(float2), 256);
  off += L.slot_bytes * (size_t)c.max_pending_updates;
  L.t64_off = off;
  L.t64_bytes = align_up((size_t)c.n_gates * c.n_doppler * sizeof(double2), 256);
  off += L.t64_bytes;
  L.tw_off = off;
  off += align_up((size_t)c.n_doppler * sizeof(float2), 256);
  L.ctr_off = off;
  off += align_up(kNumCounters * sizeof(unsigned int), 256);
  L.stage_off = off;
  L.stage_buf_bytes = align_up((size_t)c.host_stage_scatterers * sizeof(float), 256) * 7;
  off += 2 * L.stage_buf_bytes;
  L.iq_off = off;
  L.iq_bytes = align_up((size_t)c.host_stage_pulses * c.n_gates * sizeof(float2), 256);
  off += L.iq_bytes;
  L.total = off;
  return L;
}

const char* check_config(const sim_config* c) {
  if (!c) return "cfg is NULL";
  if (c->struct_size != sizeof(sim_config)) return "cfg.struct_size != sizeof(sim_config) (ABI mismatch)";
  if (c->n_gates < 1 || c->n_gates > 1024) return "n_gates must be in 1..1024";
  {
    int radix[kSynMaxPass], n_pass = 0;
    if (c->n_doppler < 16 || c->n_doppler > 4096 || !synth_factor(c->n_doppler, radix, &n_pass))
      return "n_doppler must be in 16..4096 with no prime factor other than 2, 3 and 5";
  }
  if (c->pulses_per_update < 1) return "pulses_per_update must be >= 1";
  if (c->max_pending_updates < 2) return "max_pending_updates must be >= 2";
  if (c->weight_mode != SIM_W_SQRT && c->weight_mode != SIM_W_LINEAR) return "unknown weight_mode";
  if (c->doppler_mode != SIM_DOPPLER_ANALYTIC && c->doppler_mode != SIM_DOPPLER_PULSE_PAIR) return "unknown doppler_mode";
  if (!(c->wavelength_m > 0) || !std::isfinite(c->wavelength_m)) return "wavelength_m must be > 0";
  if (!(c->prf_hz > 0) || !std::isfinite(c->prf_hz)) return "prf_hz must be > 0";
  if (!(c->gate_spacing_m > 0) || !std::isfinite(c->gate_spacing_m)) return "gate_spacing_m must be > 0";
  if (!(c->antenna_alpha >= 0) || !std::isfinite(c->antenna_alpha)) return "antenna_alpha must be >= 0";
  if (c->host_stage_scatterers < 0 || c->host_stage_pulses < 0) return "host staging sizes must be >= 0";
  if (c->host_stage_scatterers % 4) return "host_stage_scatterers must be a multiple of 4";
  if (c->device < 0) return "device must be >= 0";
  return nullptr;
}

}  // namespace

struct sim_handle {
  sim_config cfg;
  Layout lay;
  unsigned char* ws;
  cudaStream_t stream;
  cudaStream_t copy_stream;      // only with host staging
  cudaEvent_t ev_copied[2];      // staging buffer b filled
  cudaEvent_t ev_consumed[2];    // staging buffer b consumed by the kernel
  bool stage_used[2];
  int sm_count;
  size_t smem_optin;
  // stream state
  int64_t n_updates;             // spectra started so far
  int64_t pulses_emitted;
  // tuning
  int opt_variant, opt_blocks, opt_window, opt_index_path, opt_guard;
  int64_t opt_superchunk;
  int opt_ncw;                      // warps per block
  int ws_W, ws_stages, ws_blocks_per_sm;   // planned window width, ring depth, resident blocks per SM
  int opt_scatter;
  int opt_il;
  int opt_pt, opt_epoch;            // scatterers per lane per chunk; scatterers per fixed-point epoch
  size_t smem_per_sm;
  // stats
  // tabulated antenna pattern (device table of the caller; nullptr: analytic gain)
  const float2* lut;
  int lut_nu, lut_nv;
  double lut_u0, lut_du, lut_v0, lut_dv;
  uint64_t launches, scatterers_seen;
  std::string err;
};

namespace {

// Makes the handle's device current for the duration of a call and restores the caller's afterwards.
struct DeviceGuard {
  int prev = -1;
  bool switched = false;
  explicit DeviceGuard(int device) {
    if (cudaGetDevice(&prev) == cudaSuccess && prev != device) switched = cudaSetDevice(device) == cudaSuccess;
  }
  ~DeviceGuard() {
    if (switched) cudaSetDevice(prev);
  }
};

int fail(sim_handle* h, int code, const std::string& msg) {
  if (h) h->err = msg; else g_create_error = msg;
  return code;
}
int cuda_fail(sim_handle* h, cudaError_t e, const char* what) {
  return fail(h, SIM_ERR_CUDA, std::string(what) + ": " + cudaGetErrorString(e));
}

float2* slot_ptr(sim_handle* h, int64_t u) {
  return reinterpret_cast<float2*>(h->ws + h->lay.ring_off + (size_t)(u % h->cfg.max_pending_updates) * h->lay.slot_bytes);
}
unsigned int* counters(sim_handle* h) { return reinterpret_cast<unsigned int*>(h->ws + h->lay.ctr_off); }

int64_t oldest_needed(const sim_handle* h) { return h->pulses_emitted / h->cfg.pulses_per_update; }

bool misaligned(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) != 0; }

int check_scatterers(sim_handle* h, const sim_scatterers* s, bool device_ptrs) {
  if (!s) return fail(h, SIM_ERR_INVALID_ARG, "scatterers is NULL");
  if (s->n == 0) return SIM_OK;
  const float* a[7] = {s->x, s->y, s->z, s->vx, s->vy, s->vz, s->s0dA};
  for (int i = 0; i < 7; ++i) {
    if (!a[i]) return fail(h, SIM_ERR_INVALID_ARG, "a scatterer array is NULL");
    if (device_ptrs && misaligned(a[i])) return fail(h, SIM_ERR_INVALID_ARG, "scatterer arrays must be 16-byte aligned");
  }
  return SIM_OK;
}

int check_sat(sim_handle* h, const sim_sat_state* sat) {
  if (!sat) return fail(h, SIM_ERR_INVALID_ARG, "sat_state is NULL");
  const double b2 = sat->boresight[0] * sat->boresight[0] + sat->boresight[1] * sat->boresight[1] +
                    sat->boresight[2] * sat->boresight[2];
  if (!(b2 > 0) || !std::isfinite(b2)) return fail(h, SIM_ERR_INVALID_ARG, "boresight must be a finite non-zero vector");
  for (int i = 0; i < 3; ++i)
    if (!std::isfinite(sat->pos[i]) || !std::isfinite(sat->vel[i])) return fail(h, SIM_ERR_INVALID_ARG, "sat_state is not finite");
  if (!std::isfinite(sat->range_gate0_m)) return fail(h, SIM_ERR_INVALID_ARG, "range_gate0_m is not finite");
  return SIM_OK;
}

// Constants of the sqrt/divide-free index path and the decision whether it is valid for this geometry
// (error bounds that the guard band must cover).
void fast_path_constants(const sim_handle* h, const sim_sat_state* sat, AccParams& p) {
  const double rg0 = sat->range_gate0_m, dR = h->cfg.gate_spacing_m, lam = h->cfg.wavelength_m;
  const int G = h->cfg.n_gates;
  p.guard = h->opt_guard;
  p.guard_k = h->opt_guard;
  p.fast_ok = 0;
  p.pp_ok = 0;
  {  // frac(rg0 * 2 / lambda) to ~1e-17 cycles: product split into rounded part + exact residual
    const double c = 2.0 / lam, q = rg0 * c, qe = std::fma(rg0, c, -q);
    p.fr0 = (q - std::floor(q)) + qe;
    p.fr0m = p.fr0 + 402653184.0;   // 1.5 * 2^28
  }
  if (!(rg0 > 0)) return;
  const double margin = 0.01 * dR + 1e-9 * rg0;
  const double d_lo = -dR - margin, d_hi = G * dR + margin;
  const double dmax = std::fmax(-d_lo, d_hi), emax = dmax / rg0, rmax = rg0 + d_hi;
  if (!(rg0 + d_lo > 0) || !(emax < 1.0 / 1024.0)) return;
  p.inv_2rg0 = 0.5 / rg0;
  const double c = 2.0 / lam;
  const bool phase_ok = (G + 2) * dR * c < 134217728.0;   // 2^27: the magic-number fraction needs |q| < 2^28
  {  // polynomial index path (scatter_math.cuh), x = u / rg0^2 <= ~2 emax
    const double r2 = rg0 * rg0, gd = p.guard / (double)(1 << kFracBits);
    p.neg_rg0sq = -r2;
    p.g1 = 1.0 / (2.0 * rg0 * dR);
    p.g2 = -1.0 / (8.0 * rg0 * r2 * dR);
    p.g3 = 1.0 / (16.0 * rg0 * r2 * r2 * dR);
    p.j0 = p.cD / rg0;
    p.j1 = -p.cD / (2.0 * rg0 * r2);
    p.j2 = 3.0 * p.cD / (8.0 * rg0 * r2 * r2);
    p.cq = dR * c;
    const double mg = 0.5 * gd;                                   // window margin, gates (half a guard band)
    const double wl = -dR * (1.0 + mg), wh = dR * (G + mg);
    p.uw_lo = wl * (2.0 * rg0 + wl);
    p.uw_hi = wh * (2.0 * rg0 + wh);
    const double x = 2.2 * emax;
    const double eg = 0.04 * x * x * x * x * rg0 / dR + 4.0 * std::ldexp(r2, -52) / (2.0 * rg0 * dR) + 1e-13 * (G + 2);
    const double ek = 1024.0 * (0.32 * x * x * x + 1e-14);
    if (gd >= 4.0 * eg && gd >= 4.0 * ek && phase_ok && G + 2 < 2048) p.fast_ok = 1;
  }
  {  // pulse-pair polynomial path (scatter_math.cuh, kIdxFastPulsePair).  The canonical R' - R carries the rounding of
     // two square roots of ~rmax (each within 2 ulp of the exact root): up to 4 * 2^-53 * rmax * 2N / lambda bins of
     // noise that the (accurate) fast value does not share; the Doppler guard band is 1.5 x that bound.  Series and
     // roundings of the fast value itself: 1024 * (e^3 + 1e-14), e <= 2.2 emax.
    const double cP_abs = 2.0 * (double)h->cfg.n_doppler / lam;
    const double noise = 4.0 * std::ldexp(rmax, -53) * cP_abs;
    const double x = 2.2 * emax;
    const double own = 1024.0 * (x * x * x + 1e-14);
    const double need = 1.5 * noise + 4.0 * own;
    int gk = (int)std::ceil(need * (double)(1 << kFracBits));
    if (gk < p.guard) gk = p.guard;
    p.two_dR = 2.0 * dR;
    p.cP_2rg0 = p.cP * p.inv_2rg0;
    p.pp_ok = (p.fast_ok && gk <= (1 << (kFracBits - 3))) ? 1 : 0;   // the gate half of the bound is the analytic one
    p.guard_k = h->cfg.doppler_mode == SIM_DOPPLER_PULSE_PAIR ? gk : p.guard;
  }
}

int acc_blocks(const sim_handle* h) {
  if (h->opt_blocks > 0) return h->opt_blocks;
  return h->sm_count * (h->ws_blocks_per_sm > 0 ? h->ws_blocks_per_sm : 1);
}

// Per-variant defaults (measured on the 268M and 16.8M configs, profiles/).
void variant_defaults(sim_handle* h) {
  h->opt_ncw = 8; h->opt_pt = 4; h->opt_il = 4; h->opt_epoch = 8191;
}

// Window width, ring depth and resident blocks per SM of the tile kernels for the shared memory there is.
cudaError_t plan_ws(sim_handle* h) {
  if (h->opt_variant == 0) {   // the reference kernel has no tile
    h->ws_W = 1; h->ws_stages = 2; h->ws_blocks_per_sm = 8;
    return cudaSuccess;
  }
  const int G = h->cfg.n_gates, N = h->cfg.n_doppler, ncw = h->opt_ncw, pt = h->opt_pt;
  if (!acc_supported(ncw, pt, h->opt_il)) return cudaErrorInvalidValue;
  auto smem = [&](int g, int w, int st) { return acc_smem_bytes(g, w, ncw, pt, st); };
  const int target = ncw <= 8 ? 2 : 1;                              // blocks per SM the register budget allows
  size_t budget = h->smem_per_sm / target;
  budget = budget > 2048 ? budget - 2048 : 0;                       // 1 KB reserved per block + static shared memory
  if (budget > h->smem_optin - 4096) budget = h->smem_optin - 4096;   // the kernels' static shared memory (< 3 KB) counts against the opt-in limit
  const size_t stage = smem(0, 0, 1) - smem(0, 0, 0);
  const int st = 2;   // every lane copies one chunk ahead of its reads: two stages
  int want = h->opt_window > 0 ? h->opt_window : 20;
  if (want > N) want = N;
  auto widest = [&](size_t bytes) {
    int v = want;
    while (v > 1 && smem(G, v, 0) + st * stage > bytes) --v;
    return v;
  };
  int w = widest(budget);
  if (target == 2 && w < 4 && want >= 4) {
    // Very many gates (beyond ~440): two blocks per SM leave no room for even a 4-bin window, and every contribution
    // would go to the global fp64 reductions (measured on the 16.8M patch, G = 512 / 1024: 621 / 470 us per update).
    // One block per SM with all of the SM's shared memory holds a window again (166 / 175 us).  A 4-bin window at two
    // blocks per SM, where it fits (G = 192, 256: 117 us), beats a 20-bin window at one block (174-179 us), so the
    // re-plan is taken only when the two-block plan has no window at all.
    size_t one = h->smem_per_sm > 2048 ? h->smem_per_sm - 2048 : 0;
    if (one > h->smem_optin - 4096) one = h->smem_optin - 4096;
    const int w1 = widest(one);
    if (w1 > w) w = w1;
  }
  if (h->opt_window == 0 && acc_row_stride(w) <= N) w = acc_row_stride(w);   // the padding columns of a row are free
  h->ws_W = w;
  h->ws_stages = st;
  int b = 1;
  cudaError_t e = acc_blocks_per_sm(G, w, ncw, pt, h->opt_il, st, &b);
  h->ws_blocks_per_sm = b > 0 ? b : 1;
  return e;
}

AccParams make_acc_params(sim_handle* h, const sim_scatterers* s, const sim_sat_state* sat, float2* T) {
  AccParams p{};
  p.x = s->x; p.y = s->y; p.z = s->z; p.vx = s->vx; p.vy = s->vy; p.vz = s->vz; p.s0dA = s->s0dA;
  p.n = s->n;
  p.sx = sat->pos[0]; p.sy = sat->pos[1]; p.sz = sat->pos[2];
  p.svx = sat->vel[0]; p.svy = sat->vel[1]; p.svz = sat->vel[2];
  p.rg0 = sat->range_gate0_m;
  // host constants of the canonical sequence, each by exactly this expression
  p.inv_dR = 1.0 / h->cfg.gate_spacing_m;
  p.two_over_lambda = 2.0 / h->cfg.wavelength_m;
  p.cD = (-2.0 * (double)h->cfg.n_doppler) / (h->cfg.wavelength_m * h->cfg.prf_hz);
  p.doppler_mode = h->cfg.doppler_mode;
  p.pri = 1.0 / h->cfg.prf_hz;
  p.cP = (-2.0 * (double)h->cfg.n_doppler) / h->cfg.wavelength_m;
  fast_path_constants(h, sat, p);
  const double bn = std::sqrt(sat->boresight[0] * sat->boresight[0] + sat->boresight[1] * sat->boresight[1] +
                              sat->boresight[2] * sat->boresight[2]);
  p.sxh = (float)sat->pos[0];
  p.syh = (float)sat->pos[1];
  p.szh = (float)sat->pos[2]; p.szl = (float)(sat->pos[2] - (double)p.szh);
  p.neg_alpha_log2e = (float)(-h->cfg.antenna_alpha * 1.4426950408889634);
  {  // orthonormal basis (e1, e2) of the plane normal to the boresight: sin^2 = ((d.e1)^2 + (d.e2)^2) / R^2.
     // e1 = along track (reading R9: the u axis of the tabulated pattern), e2 = b x e1; when the velocity is parallel
     // to the boresight any basis serves the analytic gain (the tabulated one is refused by check_lut_frame)
    const double b[3] = {sat->boresight[0] / bn, sat->boresight[1] / bn, sat->boresight[2] / bn};
    const double vb = sat->vel[0] * b[0] + sat->vel[1] * b[1] + sat->vel[2] * b[2];
    double e1[3] = {sat->vel[0] - vb * b[0], sat->vel[1] - vb * b[1], sat->vel[2] - vb * b[2]};
    double n1 = std::sqrt(e1[0] * e1[0] + e1[1] * e1[1] + e1[2] * e1[2]);
    const double vn = std::sqrt(sat->vel[0] * sat->vel[0] + sat->vel[1] * sat->vel[1] + sat->vel[2] * sat->vel[2]);
    if (!(n1 > 1e-9 * vn) || !(n1 > 0)) {
      int ax = 0;
      if (std::fabs(b[1]) < std::fabs(b[ax])) ax = 1;
      if (std::fabs(b[2]) < std::fabs(b[ax])) ax = 2;
      double a[3] = {0, 0, 0};
      a[ax] = 1.0;
      e1[0] = b[1] * a[2] - b[2] * a[1]; e1[1] = b[2] * a[0] - b[0] * a[2]; e1[2] = b[0] * a[1] - b[1] * a[0];
      n1 = std::sqrt(e1[0] * e1[0] + e1[1] * e1[1] + e1[2] * e1[2]);
    }
    for (double& v : e1) v /= n1;
    const double e2[3] = {b[1] * e1[2] - b[2] * e1[1], b[2] * e1[0] - b[0] * e1[2], b[0] * e1[1] - b[1] * e1[0]};
    p.e1x = (float)e1[0]; p.e1y = (float)e1[1]; p.e1z = (float)e1[2];
    p.e2x = (float)e2[0]; p.e2y = (float)e2[1]; p.e2z = (float)e2[2];
    p.e1c = (float)-((double)p.e1x * sat->pos[0] + (double)p.e1y * sat->pos[1] + (double)p.e1z * sat->pos[2]);
    p.e2c = (float)-((double)p.e2x * sat->pos[0] + (double)p.e2y * sat->pos[1] + (double)p.e2z * sat->pos[2]);
    const double rg0 = sat->range_gate0_m, dRf = h->cfg.gate_spacing_m / (double)(1 << kFracBits);
    p.a0 = (float)(1.0 / (rg0 * rg0));
    p.a1 = (float)(-2.0 * dRf / (rg0 * rg0 * rg0));
    p.a2 = (float)(3.0 * dRf * dRf / (rg0 * rg0 * rg0 * rg0));
    p.w_scale = (float)(1.0 / (double)(1 << kFracBits));
  }
  p.lut = h->lut;
  p.lut_nu = h->lut_nu; p.lut_nv = h->lut_nv;
  p.lut_u0 = (float)h->lut_u0; p.lut_v0 = (float)h->lut_v0;
  p.lut_inv_du = h->lut ? (float)(1.0 / h->lut_du) : 0.0f;
  p.lut_inv_dv = h->lut ? (float)(1.0 / h->lut_dv) : 0.0f;
  p.G = h->cfg.n_gates;
  p.N = h->cfg.n_doppler;
  p.T = T;
  p.T64 = reinterpret_cast<double2*>(h->ws + h->lay.t64_off);
  p.counters = counters(h);
  const int blocks = acc_blocks(h);
  const int ch = acc_chunk(h->opt_ncw, h->opt_pt);
  unsigned long long sc = (unsigned long long)h->opt_superchunk;
  if (sc == 0) {
    // aim at >= 8 scheduling units per block, between one chunk and 16K scatterers
    sc = 16384;
    while (sc > (unsigned long long)ch && s->n / sc < (unsigned long long)blocks * 8) sc >>= 1;
  }
  // chunks per fixed-point epoch: as many as the epoch length allows, but a small input is cut into enough
  // scheduling units (whole epochs) to give every resident block some work
  int ec = h->opt_epoch / ch > 0 ? h->opt_epoch / ch : 1;
  {
    const unsigned long long fair = s->n / ((unsigned long long)ch * (unsigned long long)blocks * 2ull);
    if (fair < (unsigned long long)ec) ec = fair > 0 ? (int)fair : 1;
  }
  p.W = h->ws_W;
  p.row_words = acc_row_stride(p.W);
  p.plane_words = acc_plane_words(h->cfg.n_gates, p.W);
  p.stages = h->ws_stages;
  {  // epoch of L scatterers: L adds of at most 2^fx_cap (+ rounding) per cell stay below 2^31
    const int L = ec * ch;
    int lg = 0;
    while ((1 << lg) < L + 1) ++lg;
    p.fx_cap = 31 - lg;
    p.fx_target = p.fx_cap - 2 < 16 ? p.fx_cap - 2 : 16;
  }
  p.epoch_chunks = ec;
  const unsigned long long unit = (unsigned long long)ch * p.epoch_chunks;   // scheduling unit = whole epochs: a jump never splits one
  if (sc > (1ull << 30)) sc = 1ull << 30;   // the kernels count the scatterers of a unit in 32 bits
  sc = (sc + unit - 1) / unit * unit;
  p.superchunk = sc;
  {  // The last round of work goes in shorter units (half an epoch), in input order: the blocks then finish within
     // a short unit of each other instead of a long one (measured on the 16.8M patch: the tail of a launch was about half
     // a unit, 7 us of 121).  Not when the caller fixed the unit size, and never more than a quarter of the input.
    const unsigned long long n_full = s->n / sc;
    unsigned long long tail_big = 0;
    if (h->opt_superchunk == 0 && ec >= 3) {
      tail_big = (unsigned long long)blocks < n_full / 4 ? (unsigned long long)blocks : n_full / 4;
    }
    const unsigned long long n_big = n_full - tail_big;
    const int ec_small = tail_big ? (ec + 1) / 2 : ec;   // (half, a third or a quarter of an epoch, and one round or two, measure alike within 1-2 %)
    p.sc_small = tail_big ? (unsigned long long)ch * ec_small : sc;
    p.tail_start = n_big * sc;
    const unsigned long long n_small = (s->n - p.tail_start + p.sc_small - 1) / p.sc_small;
    p.n_big = (unsigned)n_big;
    p.n_units = (unsigned)(n_big + n_small);
    // scattered visiting order of the whole units: dark and illuminated parts of the scene are in flight at the same
    // time, so the DRAM-bound and the compute-bound phases overlap instead of alternating
    unsigned long long stride = 1;
    if (h->opt_scatter && n_big > 2) {
      stride = (unsigned long long)((double)n_big * 0.6180339887498949);
      auto gcd = [](unsigned long long a, unsigned long long b) { while (b) { const unsigned long long t = a % b; a = b; b = t; } return a; };
      while (stride > 1 && gcd(stride, n_big) != 1) --stride;
      if (stride < 1) stride = 1;
    }
    p.sc_stride = stride;
  }
  p.index_path = h->opt_index_path;
  return p;
}

// The geometry every kernel's fp32 amplitude series is budgeted for (1/R^2 to second order about rg0): window depth
// <= 0.6 % of rg0 keeps its truncation below 1e-6.
int check_geometry(sim_handle* h, const sim_sat_state* sat) {
  const double rg0 = sat->range_gate0_m, depth = (h->cfg.n_gates + 2) * h->cfg.gate_spacing_m;
  if (!(rg0 > 0)) return fail(h, SIM_ERR_BAD_CONFIG, "range_gate0_m must be > 0");
  if (!(depth / rg0 <= 6e-3)) return fail(h, SIM_ERR_BAD_CONFIG, "gate window deeper than 0.6 % of range_gate0_m: outside the range of the amplitude series");
  return SIM_OK;
}

// One accumulation launch into the fp64 accumulator.
int do_accumulate(sim_handle* h, const sim_scatterers* d_scat, const sim_sat_state* sat, float2* T) {
  AccParams p = make_acc_params(h, d_scat, sat, T);
  const int blocks = acc_blocks(h);
  int l = 0;
  cudaError_t e = h->opt_variant == 0 ? launch_reference(p, h->sm_count, h->stream, &l)
                                      : launch_accumulate(p, h->opt_ncw, h->opt_pt, h->opt_il, blocks, false, h->stream, &l);
  h->launches += l;
  if (e != cudaSuccess) return cuda_fail(h, e, "accumulate launch");
  return SIM_OK;
}

// fp64 accumulator -> spectrum slot (assign, or add for SIM_ACC_APPEND).
int do_finalize(sim_handle* h, float2* T, bool add) {
  int l = 0;
  cudaError_t e = launch_finalize(reinterpret_cast<double2*>(h->ws + h->lay.t64_off), T, h->cfg.n_gates * h->cfg.n_doppler, add,
                                  h->stream, &l);
  h->launches += l;
  if (e != cudaSuccess) return cuda_fail(h, e, "finalize launch");
  return SIM_OK;
}

// After a failed launch sequence: whatever reached the fp64 accumulator is discarded (best effort).
void scrub_accumulator(sim_handle* h) {
  cudaMemsetAsync(h->ws + h->lay.t64_off, 0, h->lay.t64_bytes, h->stream);
}

// A tabulated pattern needs its along-track axis (reading R9).
int check_lut_frame(sim_handle* h, const sim_sat_state* sat) {
  if (!h->lut) return SIM_OK;
  const double bn2 = sat->boresight[0] * sat->boresight[0] + sat->boresight[1] * sat->boresight[1] + sat->boresight[2] * sat->boresight[2];
  const double vb = sat->vel[0] * sat->boresight[0] + sat->vel[1] * sat->boresight[1] + sat->vel[2] * sat->boresight[2];
  const double v2 = sat->vel[0] * sat->vel[0] + sat->vel[1] * sat->vel[1] + sat->vel[2] * sat->vel[2];
  const double perp2 = v2 - vb * vb / bn2;
  if (!(perp2 > 1e-18 * v2) || !(v2 > 0))
    return fail(h, SIM_ERR_INVALID_ARG, "antenna table set and satellite velocity parallel to the boresight: no along-track axis");
  return SIM_OK;
}

// Common front of the two accumulate entry points: validates everything and says which slot the update uses.
// Changes NOTHING in the handle: the caller commits (n_updates, scatterers_seen) only after its launches succeeded.
int begin_update(sim_handle* h, const sim_scatterers* s, const sim_sat_state* sat, uint32_t flags,
                 bool device_ptrs, float2** T) {
  if (!h) return fail(nullptr, SIM_ERR_INVALID_ARG, "handle is NULL");
  if (flags & ~SIM_ACC_APPEND) return fail(h, SIM_ERR_INVALID_ARG, "unknown accumulate flag");
  int rc = check_scatterers(h, s, device_ptrs);
  if (rc) return rc;
  rc = check_sat(h, sat);
  if (rc) return rc;
  rc = check_geometry(h, sat);
  if (rc) return rc;
  rc = check_lut_frame(h, sat);
  if (rc) return rc;
  if (flags & SIM_ACC_APPEND) {
    if (h->n_updates == 0) return fail(h, SIM_ERR_INVALID_ARG, "SIM_ACC_APPEND before any update");
    *T = slot_ptr(h, h->n_updates - 1);
    return SIM_OK;
  }
  if (h->n_updates - oldest_needed(h) >= h->cfg.max_pending_updates)
    return fail(h, SIM_ERR_OVERFLOW, "ring full: synthesize pulses before accumulating another update");
  *T = slot_ptr(h, h->n_updates);
  return SIM_OK;
}

int plan_synthesis(sim_handle* h, int64_t n_pulses, const void* iq, uint32_t flags, int64_t* s_first,
                   int64_t* s_last) {
  if (!h) return fail(nullptr, SIM_ERR_INVALID_ARG, "handle is NULL");
  if (flags & ~SIM_SYN_FINAL) return fail(h, SIM_ERR_INVALID_ARG, "unknown synthesize flag");
  if (n_pulses < 0) return fail(h, SIM_ERR_INVALID_ARG, "n_pulses < 0");
  if (n_pulses == 0) return SIM_OK;
  if (!iq) return fail(h, SIM_ERR_INVALID_ARG, "iq buffer is NULL");
  const int64_t P = h->cfg.pulses_per_update;
  *s_first = h->pulses_emitted / P;
  *s_last = (h->pulses_emitted + n_pulses - 1) / P;
  if (*s_last >= h->n_updates) return fail(h, SIM_ERR_NOT_READY, "spectrum of the last segment has not been accumulated");
  if (*s_last + 1 >= h->n_updates && !(flags & SIM_SYN_FINAL))
    return fail(h, SIM_ERR_NOT_READY, "successor spectrum missing (accumulate it or pass SIM_SYN_FINAL)");
  return SIM_OK;
}

int do_synthesize(sim_handle* h, int64_t n_pulses, float2* d_iq, int64_t s_first, int64_t s_last) {
  SynParams p{};
  p.ring = reinterpret_cast<const float2*>(h->ws + h->lay.ring_off);
  p.slot_stride = h->lay.slot_bytes / sizeof(float2);
  p.cap = h->cfg.max_pending_updates;
  p.tw = reinterpret_cast<const float2*>(h->ws + h->lay.tw_off);
  p.iq = d_iq;
  p.x0 = h->pulses_emitted;
  p.n_pulses = n_pulses;
  p.seg0 = s_first;
  p.n_spectra = h->n_updates;
  p.G = h->cfg.n_gates;
  p.N = h->cfg.n_doppler;
  p.P = h->cfg.pulses_per_update;
  p.n_segments = s_last - s_first + 1;
  synth_plan(p.N, p.G, p.P, p.n_segments, h->sm_count, &p.GT, &p.seg_per_block);
  p.weight_mode = h->cfg.weight_mode;
  int l = 0;
  cudaError_t e = launch_synthesize(p, h->stream, &l);
  h->launches += l;
  if (e != cudaSuccess) return cuda_fail(h, e, "synthesize launch");
  h->pulses_emitted += n_pulses;
  return SIM_OK;
}

}  // namespace

extern "C" {

int sim_workspace_bytes(const sim_config* cfg, size_t* out_bytes) {
  if (!out_bytes) return fail(nullptr, SIM_ERR_INVALID_ARG, "out_bytes is NULL");
  if (const char* m = check_config(cfg)) return fail(nullptr, cfg ? SIM_ERR_BAD_CONFIG : SIM_ERR_INVALID_ARG, m);
  *out_bytes = make_layout(*cfg).total;
  return SIM_OK;
}

int sim_create(const sim_config* cfg, void* d_workspace, size_t bytes, void* cuda_stream, sim_handle** out) {
  if (!out) return fail(nullptr, SIM_ERR_INVALID_ARG, "out is NULL");
  *out = nullptr;
  if (const char* m = check_config(cfg)) return fail(nullptr, cfg ? SIM_ERR_BAD_CONFIG : SIM_ERR_INVALID_ARG, m);
  const Layout lay = make_layout(*cfg);
  if (!d_workspace) return fail(nullptr, SIM_ERR_WORKSPACE, "workspace is NULL");
  if (reinterpret_cast<uintptr_t>(d_workspace) & 255u) return fail(nullptr, SIM_ERR_WORKSPACE, "workspace must be 256-byte aligned");
  if (bytes < lay.total) return fail(nullptr, SIM_ERR_WORKSPACE, "workspace smaller than sim_workspace_bytes");
  int n_dev = 0;
  cudaError_t e = cudaGetDeviceCount(&n_dev);
  if (e != cudaSuccess) return cuda_fail(nullptr, e, "cudaGetDeviceCount");
  if (cfg->device >= n_dev) return fail(nullptr, SIM_ERR_BAD_CONFIG, "cfg.device is not a CUDA device of this process");
  DeviceGuard guard(cfg->device);   // the caller's current device is restored on return
  sim_handle* h = new (std::nothrow) sim_handle();
  if (!h) return fail(nullptr, SIM_ERR_INVALID_ARG, "out of host memory");
  h->cfg = *cfg;
  h->lay = lay;
  h->ws = static_cast<unsigned char*>(d_workspace);
  h->stream = static_cast<cudaStream_t>(cuda_stream);
  h->copy_stream = nullptr;
  h->ev_copied[0] = h->ev_copied[1] = h->ev_consumed[0] = h->ev_consumed[1] = nullptr;
  h->stage_used[0] = h->stage_used[1] = false;
  h->n_updates = 0;
  h->pulses_emitted = 0;
  h->lut = nullptr;
  h->lut_nu = h->lut_nv = 0;
  h->lut_u0 = h->lut_du = h->lut_v0 = h->lut_dv = 0.0;
  h->opt_variant = 4;
  variant_defaults(h);
  h->opt_scatter = 1;
  h->opt_blocks = 0;
  h->opt_window = 0;
  h->opt_index_path = 1;
  h->opt_guard = 16;
  h->opt_superchunk = 0;
  h->ws_W = 0;
  h->ws_stages = 0;
  h->ws_blocks_per_sm = 0;
  h->launches = 0;
  h->scatterers_seen = 0;
  int v = 0;
  e = cudaDeviceGetAttribute(&v, cudaDevAttrMultiProcessorCount, cfg->device);
  if (e != cudaSuccess) { sim_destroy(h); return cuda_fail(nullptr, e, "cudaDeviceGetAttribute(sm count)"); }
  h->sm_count = v;
  e = cudaDeviceGetAttribute(&v, cudaDevAttrMaxSharedMemoryPerBlockOptin, cfg->device);
  if (e != cudaSuccess) { sim_destroy(h); return cuda_fail(nullptr, e, "cudaDeviceGetAttribute(smem optin)"); }
  h->smem_optin = (size_t)v;
  if (cfg->host_stage_scatterers > 0 || cfg->host_stage_pulses > 0) {
    e = cudaStreamCreateWithFlags(&h->copy_stream, cudaStreamNonBlocking);
    if (e != cudaSuccess) { h->copy_stream = nullptr; sim_destroy(h); return cuda_fail(nullptr, e, "cudaStreamCreate(copy)"); }
    for (int b = 0; b < 2; ++b) {
      e = cudaEventCreateWithFlags(&h->ev_copied[b], cudaEventDisableTiming);
      if (e == cudaSuccess) e = cudaEventCreateWithFlags(&h->ev_consumed[b], cudaEventDisableTiming);
      if (e != cudaSuccess) { sim_destroy(h); return cuda_fail(nullptr, e, "cudaEventCreate"); }
    }
  }
  e = cudaDeviceGetAttribute(&v, cudaDevAttrMaxSharedMemoryPerMultiprocessor, cfg->device);
  if (e != cudaSuccess) { sim_destroy(h); return cuda_fail(nullptr, e, "cudaDeviceGetAttribute(smem per SM)"); }
  h->smem_per_sm = (size_t)v;
  e = plan_ws(h);
  if (e != cudaSuccess) { sim_destroy(h); return cuda_fail(nullptr, e, "accumulation kernel occupancy query"); }
  e = synth_prepare(cfg->n_doppler, cfg->pulses_per_update);
  if (e != cudaSuccess) { sim_destroy(h); return cuda_fail(nullptr, e, "synthesis kernel shared-memory attribute"); }
  e = cudaMemsetAsync(counters(h), 0, kNumCounters * sizeof(unsigned int), h->stream);
  if (e == cudaSuccess) e = cudaMemsetAsync(h->ws + lay.t64_off, 0, lay.t64_bytes, h->stream);
  if (e != cudaSuccess) { sim_destroy(h); return cuda_fail(nullptr, e, "cudaMemsetAsync(counters, accumulator)"); }
  int l = 0;
  e = launch_twiddles(reinterpret_cast<float2*>(h->ws + lay.tw_off), cfg->n_doppler, h->stream, &l);
  h->launches += l;
  if (e != cudaSuccess) { sim_destroy(h); return cuda_fail(nullptr, e, "twiddle launch"); }
  *out = h;
  return SIM_OK;
}

int sim_accumulate_update(sim_handle* h, const sim_scatterers* d_scat, const sim_sat_state* sat, uint32_t flags) {
  DeviceGuard guard(h ? h->cfg.device : 0);
  float2* T = nullptr;
  int rc = begin_update(h, d_scat, sat, flags, true, &T);
  if (rc) return rc;
  const bool append = (flags & SIM_ACC_APPEND) != 0;
  rc = do_accumulate(h, d_scat, sat, T);
  if (rc == SIM_OK) rc = do_finalize(h, T, append);
  if (rc) {   // nothing is committed: the update was not started (or, for APPEND, the slot keeps its earlier batches)
    const std::string msg = h->err;
    scrub_accumulator(h);
    h->err = msg;
    return rc;
  }
  if (!append) ++h->n_updates;
  h->scatterers_seen += d_scat->n;
  return SIM_OK;
}

int sim_accumulate_update_host(sim_handle* h, const sim_scatterers* h_scat, const sim_sat_state* sat, uint32_t flags) {
  DeviceGuard guard(h ? h->cfg.device : 0);
  if (h && h->cfg.host_stage_scatterers <= 0) return fail(h, SIM_ERR_INVALID_ARG, "host staging disabled (cfg.host_stage_scatterers == 0)");
  float2* T = nullptr;
  int rc = begin_update(h, h_scat, sat, flags, false, &T);
  if (rc) return rc;
  const bool append = (flags & SIM_ACC_APPEND) != 0;
  const uint64_t chunk = (uint64_t)h->cfg.host_stage_scatterers;
  const size_t arr_stride = h->lay.stage_buf_bytes / 7;  // bytes between staged arrays
  const float* src[7] = {h_scat->x, h_scat->y, h_scat->z, h_scat->vx, h_scat->vy, h_scat->vz, h_scat->s0dA};
  // every chunk is accumulated into the fp64 accumulator; ONE finalize at the end moves the sum into the slot, so a
  // failure half-way leaves the slot (and the handle) as they were
  auto run = [&]() -> int {
    int b = 0;
    for (uint64_t off = 0; off < h_scat->n; off += chunk, b ^= 1) {
      const uint64_t m = (h_scat->n - off < chunk) ? h_scat->n - off : chunk;
      unsigned char* buf = h->ws + h->lay.stage_off + (size_t)b * h->lay.stage_buf_bytes;
      cudaError_t e;
      if (h->stage_used[b]) {
        e = cudaStreamWaitEvent(h->copy_stream, h->ev_consumed[b], 0);  // kernel done with this buffer
        if (e != cudaSuccess) return cuda_fail(h, e, "cudaStreamWaitEvent(consumed)");
      }
      for (int a = 0; a < 7; ++a) {
        e = cudaMemcpyAsync(buf + a * arr_stride, src[a] + off, m * sizeof(float), cudaMemcpyHostToDevice, h->copy_stream);
        if (e != cudaSuccess) return cuda_fail(h, e, "cudaMemcpyAsync(H2D scatterers)");
      }
      e = cudaEventRecord(h->ev_copied[b], h->copy_stream);
      if (e != cudaSuccess) return cuda_fail(h, e, "cudaEventRecord(copied)");
      e = cudaStreamWaitEvent(h->stream, h->ev_copied[b], 0);
      if (e != cudaSuccess) return cuda_fail(h, e, "cudaStreamWaitEvent(copied)");
      sim_scatterers d{};
      d.x = reinterpret_cast<const float*>(buf + 0 * arr_stride);
      d.y = reinterpret_cast<const float*>(buf + 1 * arr_stride);
      d.z = reinterpret_cast<const float*>(buf + 2 * arr_stride);
      d.vx = reinterpret_cast<const float*>(buf + 3 * arr_stride);
      d.vy = reinterpret_cast<const float*>(buf + 4 * arr_stride);
      d.vz = reinterpret_cast<const float*>(buf + 5 * arr_stride);
      d.s0dA = reinterpret_cast<const float*>(buf + 6 * arr_stride);
      d.n = m;
      const int rc2 = do_accumulate(h, &d, sat, T);
      if (rc2) return rc2;
      e = cudaEventRecord(h->ev_consumed[b], h->stream);
      if (e != cudaSuccess) return cuda_fail(h, e, "cudaEventRecord(consumed)");
      h->stage_used[b] = true;
    }
    return do_finalize(h, T, append);
  };
  rc = run();
  if (rc) {
    const std::string msg = h->err;
    scrub_accumulator(h);
    h->err = msg;
    return rc;
  }
  if (!append) ++h->n_updates;
  h->scatterers_seen += h_scat->n;
  return SIM_OK;
}

int sim_synthesize_pulses(sim_handle* h, int64_t n_pulses, void* d_iq, uint32_t flags) {
  DeviceGuard guard(h ? h->cfg.device : 0);
  int64_t s0 = 0, s1 = -1;
  int rc = plan_synthesis(h, n_pulses, d_iq, flags, &s0, &s1);
  if (rc || n_pulses == 0) return rc;
  if (misaligned(d_iq)) return fail(h, SIM_ERR_INVALID_ARG, "iq buffer must be 16-byte aligned");
  return do_synthesize(h, n_pulses, static_cast<float2*>(d_iq), s0, s1);
}

int sim_synthesize_pulses_host(sim_handle* h, int64_t n_pulses, void* h_iq, uint32_t flags) {
  DeviceGuard guard(h ? h->cfg.device : 0);
  if (h && n_pulses > h->cfg.host_stage_pulses) return fail(h, SIM_ERR_INVALID_ARG, "n_pulses exceeds cfg.host_stage_pulses");
  int64_t s0 = 0, s1 = -1;
  int rc = plan_synthesis(h, n_pulses, h_iq, flags, &s0, &s1);
  if (rc || n_pulses == 0) return rc;
  float2* d_iq = reinterpret_cast<float2*>(h->ws + h->lay.iq_off);
  rc = do_synthesize(h, n_pulses, d_iq, s0, s1);
  if (rc) return rc;
  cudaError_t e = cudaMemcpyAsync(h_iq, d_iq, (size_t)n_pulses * h->cfg.n_gates * sizeof(float2), cudaMemcpyDeviceToHost, h->stream);
  if (e != cudaSuccess) return cuda_fail(h, e, "cudaMemcpyAsync(D2H iq)");
  return SIM_OK;
}

int sim_regular_pulses(sim_handle* h, const sim_scatterers* d_scat, const sim_sat_state* sat, int64_t first_pulse,
                       int64_t n_pulses, void* d_iq, uint32_t flags) {
  DeviceGuard guard(h ? h->cfg.device : 0);
  if (!h) return fail(nullptr, SIM_ERR_INVALID_ARG, "handle is NULL");
  if (flags & ~SIM_ACC_APPEND) return fail(h, SIM_ERR_INVALID_ARG, "unknown regular-mode flag");
  if (n_pulses < 0 || n_pulses > (1 << 24)) return fail(h, SIM_ERR_INVALID_ARG, "n_pulses outside 0..2^24");
  if (first_pulse < -(1LL << 40) || first_pulse > (1LL << 40)) return fail(h, SIM_ERR_INVALID_ARG, "first_pulse out of range");
  int rc = check_scatterers(h, d_scat, true);
  if (rc) return rc;
  rc = check_sat(h, sat);
  if (rc) return rc;
  if (h->lut) return fail(h, SIM_ERR_BAD_CONFIG, "regular mode has no tabulated antenna pattern: clear the table first");
  if (n_pulses == 0) return SIM_OK;
  if (!d_iq) return fail(h, SIM_ERR_INVALID_ARG, "iq buffer is NULL");
  if (misaligned(d_iq)) return fail(h, SIM_ERR_INVALID_ARG, "iq buffer must be 16-byte aligned");
  AccParams p = make_acc_params(h, d_scat, sat, nullptr);
  if (!p.fast_ok) return fail(h, SIM_ERR_BAD_CONFIG, "regular mode: gate window outside the range of the polynomial gate coordinate");
  cudaError_t e = cudaSuccess;
  if (!(flags & SIM_ACC_APPEND)) {
    e = cudaMemsetAsync(d_iq, 0, (size_t)n_pulses * h->cfg.n_gates * sizeof(float2), h->stream);
    if (e != cudaSuccess) return cuda_fail(h, e, "cudaMemsetAsync(regular iq)");
  }
  int l = 0;
  e = launch_regular(p, static_cast<float2*>(d_iq), first_pulse, (int)n_pulses, h->cfg.prf_hz, h->sm_count, h->smem_optin,
                     h->stream, &l);
  h->launches += l;
  if (e == cudaErrorInvalidConfiguration) return fail(h, SIM_ERR_BAD_CONFIG, "regular mode: n_gates too large for one pulse row per thread in shared memory");
  if (e != cudaSuccess) return cuda_fail(h, e, "regular-mode launch");
  return SIM_OK;
}

int sim_burst_beams(sim_handle* h, const void* d_iq, int64_t n_pulses, int32_t burst, void* d_beams, uint32_t flags) {
  DeviceGuard guard(h ? h->cfg.device : 0);
  if (!h) return fail(nullptr, SIM_ERR_INVALID_ARG, "handle is NULL");
  if (flags) return fail(h, SIM_ERR_INVALID_ARG, "unknown burst flag");
  if (burst < 16 || burst > 128 || (burst & (burst - 1))) return fail(h, SIM_ERR_INVALID_ARG, "burst must be a power of two in 16..128");
  if (n_pulses < 0 || n_pulses % burst) return fail(h, SIM_ERR_INVALID_ARG, "n_pulses must be a non-negative multiple of burst");
  if (n_pulses == 0) return SIM_OK;
  if (!d_iq || !d_beams) return fail(h, SIM_ERR_INVALID_ARG, "iq / beams buffer is NULL");
  if (d_iq == d_beams) return fail(h, SIM_ERR_INVALID_ARG, "the transform is out of place: iq and beams must differ");
  if (misaligned(d_iq) || misaligned(d_beams)) return fail(h, SIM_ERR_INVALID_ARG, "iq / beams buffers must be 16-byte aligned");
  int logB = 0;
  while ((1 << logB) < burst) ++logB;
  int l = 0;
  const cudaError_t e = launch_burst_fft(static_cast<const float2*>(d_iq), static_cast<float2*>(d_beams), n_pulses / burst, logB,
                                         h->cfg.n_gates, h->stream, &l);
  h->launches += l;
  if (e != cudaSuccess) return cuda_fail(h, e, "burst FFT launch");
  return SIM_OK;
}

int sim_synchronize(sim_handle* h) {
  DeviceGuard guard(h ? h->cfg.device : 0);
  if (!h) return fail(nullptr, SIM_ERR_INVALID_ARG, "handle is NULL");
  cudaError_t e = cudaStreamSynchronize(h->stream);
  if (e != cudaSuccess) return cuda_fail(h, e, "cudaStreamSynchronize");
  if (h->copy_stream) {
    e = cudaStreamSynchronize(h->copy_stream);
    if (e != cudaSuccess) return cuda_fail(h, e, "cudaStreamSynchronize(copy)");
  }
  return SIM_OK;
}

int sim_destroy(sim_handle* h) {
  if (!h) return SIM_OK;
  if (h->copy_stream) {
    cudaStreamSynchronize(h->copy_stream);
    for (int b = 0; b < 2; ++b) {
      if (h->ev_copied[b]) cudaEventDestroy(h->ev_copied[b]);
      if (h->ev_consumed[b]) cudaEventDestroy(h->ev_consumed[b]);
    }
    cudaStreamDestroy(h->copy_stream);
  }
  delete h;
  return SIM_OK;
}

int sim_get_spectrum(sim_handle* h, int64_t update_index, void* d_out) {
  DeviceGuard guard(h ? h->cfg.device : 0);
  if (!h) return fail(nullptr, SIM_ERR_INVALID_ARG, "handle is NULL");
  if (!d_out) return fail(h, SIM_ERR_INVALID_ARG, "d_out is NULL");
  if (update_index < 0 || update_index >= h->n_updates || update_index < h->n_updates - h->cfg.max_pending_updates)
    return fail(h, SIM_ERR_INVALID_ARG, "spectrum not in the ring");
  cudaError_t e = cudaMemcpyAsync(d_out, slot_ptr(h, update_index), (size_t)h->cfg.n_gates * h->cfg.n_doppler * sizeof(float2),
                                  cudaMemcpyDeviceToDevice, h->stream);
  if (e != cudaSuccess) return cuda_fail(h, e, "cudaMemcpyAsync(spectrum)");
  return SIM_OK;
}

int sim_spectrum_offset(sim_handle* h, int64_t update_index, size_t* out_offset) {
  if (!h) return fail(nullptr, SIM_ERR_INVALID_ARG, "handle is NULL");
  if (!out_offset) return fail(h, SIM_ERR_INVALID_ARG, "out_offset is NULL");
  if (update_index < 0 || update_index >= h->n_updates || update_index < h->n_updates - h->cfg.max_pending_updates)
    return fail(h, SIM_ERR_INVALID_ARG, "spectrum not in the ring");
  *out_offset = (size_t)(reinterpret_cast<unsigned char*>(slot_ptr(h, update_index)) - h->ws);
  return SIM_OK;
}

int sim_debug_indices(sim_handle* h, const sim_scatterers* d_scat, const sim_sat_state* sat, int32_t* d_gate0, int32_t* d_bin) {
  DeviceGuard guard(h ? h->cfg.device : 0);
  if (!h) return fail(nullptr, SIM_ERR_INVALID_ARG, "handle is NULL");
  if (!d_scat) return fail(h, SIM_ERR_INVALID_ARG, "scatterers is NULL");
  if (d_scat->n && (!d_gate0 || !d_bin)) return fail(h, SIM_ERR_INVALID_ARG, "output arrays are NULL");
  sim_scatterers s = *d_scat;
  if (!s.s0dA) s.s0dA = s.x;  // not consulted by the index kernel
  int rc = check_scatterers(h, &s, true);
  if (rc) return rc;
  rc = check_sat(h, sat);
  if (rc) return rc;
  AccParams p = make_acc_params(h, &s, sat, nullptr);
  p.dbg_g0 = d_gate0;
  p.dbg_k = d_bin;
  int l = 0;
  // the production kernel itself, exporting its indices instead of accumulating
  cudaError_t e = launch_accumulate(p, h->opt_ncw, h->opt_pt, h->opt_il, acc_blocks(h), true, h->stream, &l);
  h->launches += l;
  if (e != cudaSuccess) return cuda_fail(h, e, "indices launch");
  return SIM_OK;
}

int sim_set_antenna_lut(sim_handle* h, const void* d_table, int32_t n_u, int32_t n_v, double u0, double du, double v0, double dv) {
  if (!h) return fail(nullptr, SIM_ERR_INVALID_ARG, "handle is NULL");
  if (!d_table) {
    h->lut = nullptr;
    return SIM_OK;
  }
  if (reinterpret_cast<uintptr_t>(d_table) & 7u) return fail(h, SIM_ERR_INVALID_ARG, "antenna table must be 8-byte aligned");
  if (n_u < 2 || n_u > 4096 || n_v < 2 || n_v > 4096) return fail(h, SIM_ERR_INVALID_ARG, "antenna table: n_u, n_v must be in 2..4096");
  if (!(du > 0) || !(dv > 0) || !std::isfinite(du) || !std::isfinite(dv) || !std::isfinite(u0) || !std::isfinite(v0))
    return fail(h, SIM_ERR_INVALID_ARG, "antenna table: steps must be > 0 and origins finite");
  h->lut = static_cast<const float2*>(d_table);
  h->lut_nu = n_u; h->lut_nv = n_v;
  h->lut_u0 = u0; h->lut_du = du; h->lut_v0 = v0; h->lut_dv = dv;
  return SIM_OK;
}

int sim_set_option(sim_handle* h, int32_t option, int64_t value) {
  DeviceGuard guard(h ? h->cfg.device : 0);
  if (!h) return fail(nullptr, SIM_ERR_INVALID_ARG, "handle is NULL");
  if (value < 0) return fail(h, SIM_ERR_INVALID_ARG, "option value < 0");
  // options that change the launch shape are re-planned; a shape the kernels do not support restores the old value
  auto replan = [&](int& field, int v, const char* what) -> int {
    const int old = field;
    field = v;
    const cudaError_t e = plan_ws(h);
    if (e != cudaSuccess) {
      field = old;
      plan_ws(h);
      cudaGetLastError();
      return fail(h, SIM_ERR_INVALID_ARG, what);
    }
    return SIM_OK;
  };
  switch (option) {
    case SIM_OPT_ACC_VARIANT: {
      if (value != 0 && value != 4) return fail(h, SIM_ERR_INVALID_ARG, "unknown accumulation variant (0 = reference kernel, 4 = production kernel)");
      const int old = h->opt_variant;
      h->opt_variant = (int)value;
      variant_defaults(h);   // warps, per-lane count and epoch length: back to the defaults
      if (plan_ws(h) != cudaSuccess) {
        h->opt_variant = old;
        plan_ws(h);
        cudaGetLastError();
        return fail(h, SIM_ERR_INVALID_ARG, "accumulation variant cannot be planned for this configuration");
      }
      return SIM_OK;
    }
    case SIM_OPT_ACC_BLOCKS:
      if (value > 65535) return fail(h, SIM_ERR_INVALID_ARG, "too many blocks");
      h->opt_blocks = (int)value;
      return SIM_OK;
    case SIM_OPT_ACC_SUPERCHUNK:
      h->opt_superchunk = value;
      return SIM_OK;
    case SIM_OPT_ACC_WINDOW_BINS:
      if (value > 2048) return fail(h, SIM_ERR_INVALID_ARG, "window bins must be <= 2048");
      return replan(h->opt_window, (int)value, "window width cannot be planned");
    case SIM_OPT_ACC_WARPS:
      return replan(h->opt_ncw, (int)value, "compute warps per block not supported by this accumulation variant");
    case SIM_OPT_ACC_PER_LANE:
      return replan(h->opt_pt, (int)value, "scatterers per lane not supported by this accumulation variant");
    case SIM_OPT_ACC_SHAPE: {
      const int ncw = (int)(value >> 16), pt = (int)((value >> 8) & 255), il = (int)(value & 255);
      const int o_ncw = h->opt_ncw, o_pt = h->opt_pt, o_il = h->opt_il;
      h->opt_ncw = ncw; h->opt_pt = pt; h->opt_il = il;
      if (plan_ws(h) != cudaSuccess) {
        h->opt_ncw = o_ncw; h->opt_pt = o_pt; h->opt_il = o_il;
        plan_ws(h);
        cudaGetLastError();
        return fail(h, SIM_ERR_INVALID_ARG, "block shape (warps, per lane, interleave) not compiled for this accumulation variant");
      }
      return SIM_OK;
    }
    case SIM_OPT_ACC_INTERLEAVE:
      return replan(h->opt_il, (int)value, "interleave not supported by this accumulation variant");
    case SIM_OPT_ACC_SCATTER:
      h->opt_scatter = value != 0;
      return SIM_OK;
    case SIM_OPT_ACC_EPOCH:
      if (value < 64 || value > 16383) return fail(h, SIM_ERR_INVALID_ARG, "scatterers per fixed-point epoch: 64..16383");
      h->opt_epoch = (int)value;
      return SIM_OK;
    case SIM_OPT_GUARD_LSB:
      if (value < 1 || value > (1 << (kFracBits - 2))) return fail(h, SIM_ERR_INVALID_ARG, "guard must be in 1..2^18");
      h->opt_guard = (int)value;
      return SIM_OK;
    case SIM_OPT_INDEX_PATH:
      if (value > 1) return fail(h, SIM_ERR_INVALID_ARG, "unknown index path");
      h->opt_index_path = (int)value;
      return SIM_OK;
    default:
      return fail(h, SIM_ERR_INVALID_ARG, "unknown option");
  }
}

int sim_get_stats(const sim_handle* h, sim_stats* out) {
  if (!h || !out) return SIM_ERR_INVALID_ARG;
  out->kernel_launches = h->launches;
  out->updates_accumulated = (uint64_t)h->n_updates;
  out->scatterers_seen = h->scatterers_seen;
  out->pulses_emitted = h->pulses_emitted;
  return SIM_OK;
}

int sim_read_counters(sim_handle* h, uint32_t* h_out, int32_t reset) {
  DeviceGuard guard(h ? h->cfg.device : 0);
  if (!h) return fail(nullptr, SIM_ERR_INVALID_ARG, "handle is NULL");
  if (!h_out) return fail(h, SIM_ERR_INVALID_ARG, "h_out is NULL");
  cudaError_t e = cudaMemcpyAsync(h_out, counters(h), 4 * sizeof(uint32_t), cudaMemcpyDeviceToHost, h->stream);
  if (e == cudaSuccess && reset) e = cudaMemsetAsync(counters(h), 0, kNumCounters * sizeof(uint32_t), h->stream);
  if (e == cudaSuccess) e = cudaStreamSynchronize(h->stream);
  if (e != cudaSuccess) return cuda_fail(h, e, "read counters");
  return SIM_OK;
}

const char* sim_last_error(const sim_handle* h) { return h ? h->err.c_str() : g_create_error.c_str(); }

}  // extern "C"

// ---------------------------------------------------------------------------------------------
// sim_accumulate_static: one update for callers that have no device workspace and cannot get one (include/sim.h).
// The scratch memory of the accumulation kernels -- the fp64 accumulator and the scheduling counters, which the other
// entry points keep in the caller's workspace -- is this file-scope array instead.  It is part of the library image:
// each device that runs anything from libsim.so holds one copy (zero-filled when the module is loaded) until exit.
// ---------------------------------------------------------------------------------------------
namespace {

constexpr size_t kStaticAccBytes = (size_t)SIM_STATIC_MAX_CELLS * sizeof(double2);   // 1 MiB
constexpr size_t kStaticCtrBytes = kNumCounters * sizeof(unsigned int);               // 256 B
static __device__ __align__(256) unsigned char g_static_scratch[kStaticAccBytes + kStaticCtrBytes];

// What the first call on a device finds out, kept for the later ones.  In host code `g_static_scratch` is only a
// stand-in for the symbol, not an address a kernel could use: the device address comes from cudaGetSymbolAddress,
// asked for with that device current.
struct StaticDevice {
  bool ready = false;
  unsigned char* scratch = nullptr;   // device address of g_static_scratch on this device
  int sm_count = 0;
  size_t smem_optin = 0, smem_per_sm = 0;
};
constexpr int kStaticMaxDevices = 64;
StaticDevice g_static_device[kStaticMaxDevices];
std::mutex g_static_mutex;

// Caller has made `device` current.  No allocation: one symbol look-up and three attribute queries.
int static_device(int device, StaticDevice* out) {
  std::lock_guard<std::mutex> lock(g_static_mutex);
  StaticDevice& d = g_static_device[device];
  if (!d.ready) {
    void* ptr = nullptr;
    cudaError_t e = cudaGetSymbolAddress(&ptr, g_static_scratch);
    if (e != cudaSuccess) return cuda_fail(nullptr, e, "cudaGetSymbolAddress(static scratch)");
    if (!ptr || (reinterpret_cast<uintptr_t>(ptr) & 255u)) return fail(nullptr, SIM_ERR_CUDA, "static scratch: unusable device address");
    int v = 0;
    e = cudaDeviceGetAttribute(&v, cudaDevAttrMultiProcessorCount, device);
    if (e != cudaSuccess) return cuda_fail(nullptr, e, "cudaDeviceGetAttribute(sm count)");
    d.sm_count = v;
    e = cudaDeviceGetAttribute(&v, cudaDevAttrMaxSharedMemoryPerBlockOptin, device);
    if (e != cudaSuccess) return cuda_fail(nullptr, e, "cudaDeviceGetAttribute(smem optin)");
    d.smem_optin = (size_t)v;
    e = cudaDeviceGetAttribute(&v, cudaDevAttrMaxSharedMemoryPerMultiprocessor, device);
    if (e != cudaSuccess) return cuda_fail(nullptr, e, "cudaDeviceGetAttribute(smem per SM)");
    d.smem_per_sm = (size_t)v;
    d.scratch = static_cast<unsigned char*>(ptr);
    d.ready = true;
  }
  *out = d;
  return SIM_OK;
}

}  // namespace

extern "C" int sim_accumulate_static(const sim_config* cfg, const sim_scatterers* d_scat, const sim_sat_state* sat,
                                     void* d_spectrum, void* cuda_stream, uint32_t flags) {
  if (const char* m = check_config(cfg)) return fail(nullptr, cfg ? SIM_ERR_BAD_CONFIG : SIM_ERR_INVALID_ARG, m);
  const size_t cells = (size_t)cfg->n_gates * (size_t)cfg->n_doppler;
  if (cells > (size_t)SIM_STATIC_MAX_CELLS)
    return fail(nullptr, SIM_ERR_BAD_CONFIG,
                "sim_accumulate_static: n_gates * n_doppler = " + std::to_string(cells) + " exceeds SIM_STATIC_MAX_CELLS = " +
                    std::to_string(SIM_STATIC_MAX_CELLS) + " (the built-in accumulator); use sim_create with a workspace");
  if (flags & ~SIM_ACC_APPEND) return fail(nullptr, SIM_ERR_INVALID_ARG, "unknown accumulate flag");
  if (!d_spectrum) return fail(nullptr, SIM_ERR_INVALID_ARG, "d_spectrum is NULL");
  if (misaligned(d_spectrum)) return fail(nullptr, SIM_ERR_INVALID_ARG, "d_spectrum must be 16-byte aligned");
  if (cfg->device >= kStaticMaxDevices) return fail(nullptr, SIM_ERR_BAD_CONFIG, "cfg.device beyond the devices this entry point keeps state for");
  int n_dev = 0;
  cudaError_t e = cudaGetDeviceCount(&n_dev);
  if (e != cudaSuccess) return cuda_fail(nullptr, e, "cudaGetDeviceCount");
  if (cfg->device >= n_dev) return fail(nullptr, SIM_ERR_BAD_CONFIG, "cfg.device is not a CUDA device of this process");
  DeviceGuard guard(cfg->device);
  StaticDevice dev;
  int rc = static_device(cfg->device, &dev);
  if (rc) return rc;

  // A handle that lives on this stack frame only and owns nothing on the device: it carries the configuration and the
  // default launch shape to the same planning and parameter code the handle-based calls use.
  sim_handle t{};
  t.cfg = *cfg;
  t.cfg.host_stage_scatterers = 0;
  t.cfg.host_stage_pulses = 0;
  t.stream = static_cast<cudaStream_t>(cuda_stream);
  t.sm_count = dev.sm_count;
  t.smem_optin = dev.smem_optin;
  t.smem_per_sm = dev.smem_per_sm;
  t.opt_variant = 4;
  variant_defaults(&t);
  t.opt_scatter = 1;
  t.opt_index_path = 1;
  t.opt_guard = 16;
  auto leave = [&](int code) {   // messages of the shared checks land in the temporary handle: hand them to the thread
    if (code) g_create_error = t.err;
    return code;
  };
  rc = check_scatterers(&t, d_scat, true);
  if (rc) return leave(rc);
  rc = check_sat(&t, sat);
  if (rc) return leave(rc);
  rc = check_geometry(&t, sat);
  if (rc) return leave(rc);
  e = plan_ws(&t);
  if (e != cudaSuccess) return leave(cuda_fail(&t, e, "accumulation kernel occupancy query"));

  float2* T = static_cast<float2*>(d_spectrum);
  AccParams p = make_acc_params(&t, d_scat, sat, T);
  p.T64 = reinterpret_cast<double2*>(dev.scratch);
  p.counters = reinterpret_cast<unsigned int*>(dev.scratch + kStaticAccBytes);
  // The array keeps what the last call left: the scheduling counters and the cells this call uses start at zero.  (The
  // accumulation kernel may start under the tail of the operation before it -- programmatic dependent launch -- but
  // reads no global memory before it has waited for that operation, so both clears are complete when it looks.)
  e = cudaMemsetAsync(p.counters, 0, kStaticCtrBytes, t.stream);
  if (e == cudaSuccess) e = cudaMemsetAsync(p.T64, 0, cells * sizeof(double2), t.stream);
  if (e != cudaSuccess) return leave(cuda_fail(&t, e, "cudaMemsetAsync(static scratch)"));
  int l = 0;
  e = launch_accumulate(p, t.opt_ncw, t.opt_pt, t.opt_il, acc_blocks(&t), false, t.stream, &l);
  if (e != cudaSuccess) return leave(cuda_fail(&t, e, "accumulate launch"));
  e = launch_finalize(p.T64, T, (int)cells, (flags & SIM_ACC_APPEND) != 0, t.stream, &l);
  if (e != cudaSuccess) return leave(cuda_fail(&t, e, "finalize launch"));
  return SIM_OK;
}
