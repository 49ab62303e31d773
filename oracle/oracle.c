/*
 * oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, fp64 CPU statement of the fast-mode hot path of arxiv 2408.11472
 * (Monnier, Camus, Hellouvry), written from /root/reference/PAPER.md and the readings
 * listed in DESIGN.md ("Readings of the paper").  It shares no code, header, table or
 * constant generator with the CUDA path under paper_2408_11472_b200/csrc/.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
 * legs may load this library.  The product path never calls it.
 *
 * Steps (paper's order and names):
 *   O1  oracle_spectrum   -- Algorithm 1 body for one update i:
 *                            C_i <- scatterers_complex_amplitudes(), R_i <- scatterers_range(),
 *                            D_i (Doppler; analytic form, reading A5), rasterize(C_i, T_fast, i, R_i, D_i)
 *                            = "sums the data D in the tensor T according to the ... coordinates"
 *                            (PAPER.md:94).  One [n_range][n_doppler] slice of T_fast.
 *   O2  oracle_idft       -- "batch of 1D iFFT on the last dimension (i.e. the Doppler dimension)
 *                            of T_fast", written out as the naive O(N^2) inverse DFT.
 *   O3  oracle_synthesize -- "Weighting the obtain time-long signals ... using equation (1)" and
 *                            "Summing the weighted time-long signals in the corresponding cells of Y"
 *                            (PAPER.md:100-101); eq. (1) at PAPER.md:61, W_i(x) = (1 - |i-x|/n_fast)^(1/2).
 *
 *   O1' oracle_spectrum_lut -- O1 with the antenna gain read from a complex table on a u-v grid by bilinear
 *                            interpolation ("all antenna patterns ... are computed and recorded on a
 *                            u-v grid.  The complex values ... at each facet are then obtained through interpolation
 *                            in the u-v grid"; reading R9 fixes the frame, the interpolation and the edge rule).
 *
 *   R   oracle_regular    -- the REGULAR mode: per-pulse complex sum of all scatterers per
 *                            range gate, surface "updated at each PRF" (reading R5).
 *
 * Pins: every function here is pinned by tests/test_oracle_pins.py (closed forms, numpy.fft
 * special case, Parseval, brute-force regular-mode sum, an independent numpy restatement); the
 * pulse-pair Doppler mode by tests/test_oracle_pulse_pair.py (the literal arg(C_{i+1} C_i^*) estimator at
 * 50 digits, the analytic f_D plus its closed-form second-order term, aliasing).
 * The integer decisions of geometry() -- a Doppler coordinate exactly half-way between two bins, a range exactly on
 * a gate boundary, the edges of the gate window and of the Doppler range -- by tests/test_oracle_decisions.py
 * (dyadic scenes that land on them without rounding, expected gates and bins as literals).
 * The table gain by tests/test_oracle_lut.py (constant table = isotropic, a table linear in u and v
 * reproduced exactly, a finely sampled Gaussian against the analytic gain within the interpolation bound,
 * mpmath closed form of single scatterers, the frame and the edge rule).
 * Parity unpinned BY THE PAPER (fixed only by DESIGN.md readings): the analytic antenna gain
 * G(theta) (A10), the tail rule for a missing successor spectrum (A3), the nearest-bin rule (A7).
 *
 * Build: gcc -std=c11 -O2 -ffp-contract=off -fopenmp -shared -fPIC oracle.c -o liboracle.so -lm
 * (-ffp-contract=off: the only fused multiply-adds are the explicit fma() calls below.)
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORACLE_W_SQRT 0   /* paper eq. (1) */
#define ORACLE_W_LINEAR 1 /* partition of unity (north_star wording), reading A1 */

#define ORACLE_DOPPLER_ANALYTIC 0   /* f_D = -2 (v_p - v_sat).u / lambda (north_star; reading A5) */
#define ORACLE_DOPPLER_PULSE_PAIR 1 /* the paper's estimator, Algorithm 1 lines 5-7 (readings A6, R4) */

#define ORACLE_GATE_NONE INT32_MIN /* scatterer touches no gate of the window / is dropped */

typedef struct {
  int32_t n_gates;           /* G */
  int32_t n_doppler;         /* N (any N >= 1 here; the naive DFT has no radix restriction) */
  int32_t pulses_per_update; /* P = n_fast */
  int32_t weight_mode;       /* ORACLE_W_* */
  double wavelength_m;       /* lambda */
  double prf_hz;             /* PRF */
  double gate_spacing_m;     /* Delta R */
  double antenna_alpha;      /* G(theta) = exp(-alpha sin^2 theta), reading A10 */
  int32_t doppler_mode;      /* ORACLE_DOPPLER_* */
} oracle_config;

typedef struct {
  double pos[3];
  double vel[3];
  double boresight[3]; /* any non-zero vector; normalised below */
  double range_gate0_m; /* range of the centre of gate 0, reading A9 */
} oracle_sat;

static const double TWO_PI = 6.283185307179586476925286766559;

/* Per-scatterer geometry of step O1.  Returns 0 when the scatterer is dropped (touches no
 * gate, non-finite range or Doppler, s0dA <= 0 is handled by the caller).  The first block
 * is the CANONICAL fp64 INDEX SEQUENCE: g0 and k must be reproduced bit for bit
 * by the GPU. */
typedef struct {
  int32_t g0, k;
  double w0, w1; /* two-gate linear weights, reading A8 */
  double R, R2, fr, kf;
  double dx, dy, dz;
} geom_t;

static int geometry(const oracle_config *c, const oracle_sat *s, double inv_dR,
                    double two_over_lambda, double cD, float xf, float yf, float zf, float vxf,
                    float vyf, float vzf, geom_t *o) {
  /* inputs widened fp32 -> fp64 exactly */
  const double dx = (double)xf - s->pos[0];
  const double dy = (double)yf - s->pos[1];
  const double dz = (double)zf - s->pos[2];
  const double R2 = fma(dz, dz, fma(dy, dy, dx * dx));
  const double R = sqrt(R2); /* R_i <- scatterers_range() */
  const double gf = (R - s->range_gate0_m) * inv_dR;
  if (!(gf >= -1.0 && gf < (double)c->n_gates)) return 0; /* neither g0 nor g0+1 in [0,G); NaN too */
  const double g0d = floor(gf);
  const double dvx = (double)vxf - s->vel[0];
  const double dvy = (double)vyf - s->vel[1];
  const double dvz = (double)vzf - s->vel[2];
  double kf;
  if (c->doppler_mode == ORACLE_DOPPLER_PULSE_PAIR) {
    /* Algorithm 1 lines 5-7: update_simulation((i n_fast + 1)/PRF), C_{i+1}, then
     * D_i = arg(C_{i+1} C_i^*) PRF / (2 pi)  (physical form of the printed formula, reading A6).
     * Scatterer and satellite both move at constant velocity over one PRI = 1/PRF, so the offset one
     * pulse later is d' = d + (v_p - v_sat)/PRF and, with C ~ exp(-i 4 pi R / lambda),
     * arg(C_{i+1} C_i^*) = -4 pi (R' - R)/lambda (mod 2 pi):  f_D N/PRF = -(2N/lambda)(R' - R) (mod N).
     * The wrap of arg() is the "mod N" of the bin (natural aliasing).  Basic IEEE operations only, so
     * that the GPU can reproduce the bin bit for bit (reading R4). */
    const double pri = 1.0 / c->prf_hz;
    const double cP = (-2.0 * (double)c->n_doppler) / c->wavelength_m;
    const double dx1 = fma(dvx, pri, dx), dy1 = fma(dvy, pri, dy), dz1 = fma(dvz, pri, dz);
    const double R1 = sqrt(fma(dz1, dz1, fma(dy1, dy1, dx1 * dx1)));
    kf = (R1 - R) * cP;
  } else {
    /* rdot = dR/dt = (v_p - v_sat).u,  u = (r_p - r_sat)/R ;  f_D = -2 rdot / lambda (reading A5) */
    const double rdot = fma(dvz, dz, fma(dvy, dy, dvx * dx)) / R;
    kf = rdot * cD; /* = f_D * N / PRF */
  }
  if (!(fabs(kf) < 1073741824.0)) return 0; /* |kf| >= 2^30 or NaN: dropped */
  const double kk = floor(kf + 0.5); /* nearest bin, ties up (reading A7) */
  const double N = (double)c->n_doppler;
  const double kmod = kk - N * floor(kk / N); /* in [0,N): negative Doppler wraps to k+N (A2) */
  const double q = R * two_over_lambda;       /* 2R/lambda, in cycles */
  o->g0 = (int32_t)g0d;
  o->kf = kf;
  o->k = (int32_t)kmod;
  o->w1 = gf - g0d;
  o->w0 = 1.0 - o->w1;
  o->R = R;
  o->R2 = R2;
  o->fr = q - floor(q); /* phase = -2 pi fr  ==  -4 pi R / lambda  (mod 2 pi) */
  o->dx = dx;
  o->dy = dy;
  o->dz = dz;
  return 1;
}

static void constants(const oracle_config *c, double *inv_dR, double *two_over_lambda, double *cD) {
  *inv_dR = 1.0 / c->gate_spacing_m;
  *two_over_lambda = 2.0 / c->wavelength_m;
  *cD = (-2.0 * (double)c->n_doppler) / (c->wavelength_m * c->prf_hz);
}

static void unit_boresight(const oracle_sat *s, double b[3]) {
  const double n = sqrt(s->boresight[0] * s->boresight[0] + s->boresight[1] * s->boresight[1] +
                        s->boresight[2] * s->boresight[2]);
  b[0] = s->boresight[0] / n;
  b[1] = s->boresight[1] / n;
  b[2] = s->boresight[2] / n;
}

/* Antenna pattern recorded on a u-v grid (reading R9).
 *   Frame: b = unit boresight; e1 = unit vector of vel - (vel.b) b (along track, normal to the boresight);
 *   e2 = b x e1.  Direction cosines of the line of sight d = r_p - r_sat:  u = d.e1 / R,  v = d.e2 / R.
 *   Table: complex64 values G[j][i] (interleaved re, im; i fastest) at u_i = u0 + i du, v_j = v0 + j dv.
 *   Gain at (u, v): bilinear interpolation between the four surrounding nodes; (u, v) outside
 *   [u0, u0 + (nu-1) du] x [v0, v0 + (nv-1) dv] (or NaN) is outside the recorded pattern: gain 0. */
typedef struct {
  const float *table; /* [nv][nu][2] */
  int32_t nu, nv;
  double u0, du, v0, dv;
} oracle_lut;

/* returns 0 when (u, v) is outside the table */
static int lut_gain(const oracle_lut *L, double u, double v, double *gre, double *gim) {
  const double fu = (u - L->u0) / L->du, fv = (v - L->v0) / L->dv;
  if (!(fu >= 0.0 && fu <= (double)(L->nu - 1) && fv >= 0.0 && fv <= (double)(L->nv - 1))) return 0;
  int i = (int)floor(fu), j = (int)floor(fv);
  if (i > L->nu - 2) i = L->nu - 2; /* the last node belongs to the last cell */
  if (j > L->nv - 2) j = L->nv - 2;
  const double a = fu - (double)i, bb = fv - (double)j;
  const float *t00 = L->table + 2 * ((int64_t)j * L->nu + i);
  const float *t01 = t00 + 2, *t10 = t00 + 2 * (int64_t)L->nu, *t11 = t10 + 2;
  const double w00 = (1.0 - a) * (1.0 - bb), w01 = a * (1.0 - bb), w10 = (1.0 - a) * bb, w11 = a * bb;
  *gre = w00 * (double)t00[0] + w01 * (double)t01[0] + w10 * (double)t10[0] + w11 * (double)t11[0];
  *gim = w00 * (double)t00[1] + w01 * (double)t01[1] + w10 * (double)t10[1] + w11 * (double)t11[1];
  return 1;
}

/* antenna frame of reading R9; returns 0 when the velocity is parallel to the boresight (no along-track axis) */
static int antenna_frame(const oracle_sat *s, const double b[3], double e1[3], double e2[3]) {
  const double vb = s->vel[0] * b[0] + s->vel[1] * b[1] + s->vel[2] * b[2];
  double t[3] = {s->vel[0] - vb * b[0], s->vel[1] - vb * b[1], s->vel[2] - vb * b[2]};
  const double n = sqrt(t[0] * t[0] + t[1] * t[1] + t[2] * t[2]);
  if (!(n > 0.0)) return 0;
  for (int i = 0; i < 3; ++i) e1[i] = t[i] / n;
  e2[0] = b[1] * e1[2] - b[2] * e1[1];
  e2[1] = b[2] * e1[0] - b[0] * e1[2];
  e2[2] = b[0] * e1[1] - b[1] * e1[0];
  return 1;
}

/* O1 for scatterers [lo,hi) into T (complex128 as [G][N][2], bin fastest).  lut == NULL: analytic gain. */
static void spectrum_range(const oracle_config *c, const oracle_sat *s, const oracle_lut *lut, int64_t lo, int64_t hi,
                           const float *x, const float *y, const float *z, const float *vx,
                           const float *vy, const float *vz, const float *s0dA, double *T) {
  double inv_dR, two_over_lambda, cD, b[3], e1[3] = {0, 0, 0}, e2[3] = {0, 0, 0};
  constants(c, &inv_dR, &two_over_lambda, &cD);
  unit_boresight(s, b);
  if (lut && !antenna_frame(s, b, e1, e2)) return;
  const int G = c->n_gates, N = c->n_doppler;
  for (int64_t p = lo; p < hi; ++p) {
    if (!(s0dA[p] > 0.0f)) continue; /* s0dA <= 0 (or NaN) contributes nothing */
    geom_t g;
    if (!geometry(c, s, inv_dR, two_over_lambda, cD, x[p], y[p], z[p], vx[p], vy[p], vz[p], &g))
      continue;
    /* antenna: sin^2(theta) = |d x b|^2 / R^2 (reading A10) */
    const double cx = g.dy * b[2] - g.dz * b[1];
    const double cy = g.dz * b[0] - g.dx * b[2];
    const double cz = g.dx * b[1] - g.dy * b[0];
    const double sin2 = (cx * cx + cy * cy + cz * cz) / g.R2;
    double gre = exp(-c->antenna_alpha * sin2), gim = 0.0;
    if (lut) { /* complex pattern value interpolated in the u-v grid */
      const double u = (g.dx * e1[0] + g.dy * e1[1] + g.dz * e1[2]) / g.R;
      const double v = (g.dx * e2[0] + g.dy * e2[1] + g.dz * e2[2]) / g.R;
      if (!lut_gain(lut, u, v, &gre, &gim)) continue;
    }
    /* C_i: sqrt(sigma0 dA) G / R^2 exp(-i 4 pi R / lambda)  (north_star) */
    const double A = sqrt((double)s0dA[p]) / g.R2;
    const double pr = cos(TWO_PI * g.fr), pi_ = -sin(TWO_PI * g.fr);
    const double re = A * (gre * pr - gim * pi_);
    const double im = A * (gre * pi_ + gim * pr);
    /* rasterize: two-gate linear split (A8), halves outside the window dropped */
    if (g.g0 >= 0 && g.g0 < G) {
      double *t = T + 2 * ((int64_t)g.g0 * N + g.k);
      t[0] += g.w0 * re;
      t[1] += g.w0 * im;
    }
    if (g.g0 + 1 >= 0 && g.g0 + 1 < G) {
      double *t = T + 2 * ((int64_t)(g.g0 + 1) * N + g.k);
      t[0] += g.w1 * re;
      t[1] += g.w1 * im;
    }
  }
}

/* O1. T is [G][N] complex128 (interleaved re,im).  accumulate != 0 adds to T (the paper's tiles,
 * PAPER.md:39); otherwise T is zeroed first.  nthreads <= 1: one plain loop.  nthreads > 1:
 * contiguous scatterer ranges per thread into private grids, summed in thread order. */
static int spectrum_any(const oracle_config *c, const oracle_sat *s, const oracle_lut *lut, int64_t n, const float *x,
                        const float *y, const float *z, const float *vx, const float *vy,
                        const float *vz, const float *s0dA, double *T, int accumulate, int nthreads) {
  if (!c || !s || !T || n < 0 || c->n_gates < 1 || c->n_doppler < 1) return -1;
  const int64_t cells = (int64_t)c->n_gates * c->n_doppler;
  if (!accumulate) memset(T, 0, (size_t)cells * 2 * sizeof(double));
  if (nthreads <= 1) {
    spectrum_range(c, s, lut, 0, n, x, y, z, vx, vy, vz, s0dA, T);
    return 1;
  }
#ifdef _OPENMP
  double *priv = (double *)calloc((size_t)nthreads * (size_t)cells * 2, sizeof(double));
  if (!priv) return -2;
#pragma omp parallel num_threads(nthreads)
  {
    const int t = omp_get_thread_num();
    const int nt = omp_get_num_threads();
    const int64_t lo = n * t / nt, hi = n * (t + 1) / nt;
    spectrum_range(c, s, lut, lo, hi, x, y, z, vx, vy, vz, s0dA, priv + (size_t)t * cells * 2);
  }
  for (int t = 0; t < nthreads; ++t)
    for (int64_t j = 0; j < cells * 2; ++j) T[j] += priv[(size_t)t * cells * 2 + j];
  free(priv);
  return nthreads;
#else
  spectrum_range(c, s, lut, 0, n, x, y, z, vx, vy, vz, s0dA, T);
  return 1;
#endif
}

int oracle_spectrum(const oracle_config *c, const oracle_sat *s, int64_t n, const float *x,
                    const float *y, const float *z, const float *vx, const float *vy,
                    const float *vz, const float *s0dA, double *T, int accumulate, int nthreads) {
  return spectrum_any(c, s, NULL, n, x, y, z, vx, vy, vz, s0dA, T, accumulate, nthreads);
}

/* O1 with the tabulated antenna pattern (reading R9).  -3: bad table or no antenna frame. */
int oracle_spectrum_lut(const oracle_config *c, const oracle_sat *s, const oracle_lut *lut, int64_t n, const float *x,
                        const float *y, const float *z, const float *vx, const float *vy,
                        const float *vz, const float *s0dA, double *T, int accumulate, int nthreads) {
  if (!lut || !lut->table || lut->nu < 2 || lut->nv < 2 || !(lut->du > 0.0) || !(lut->dv > 0.0)) return -3;
  if (s) {
    double b[3], e1[3], e2[3];
    unit_boresight(s, b);
    if (!antenna_frame(s, b, e1, e2)) return -3;
  }
  return spectrum_any(c, s, lut, n, x, y, z, vx, vy, vz, s0dA, T, accumulate, nthreads);
}

/* Indices only (canonical sequence).  g0[p] in [-1, G-1], k[p] in [0, N); a dropped scatterer
 * (out of window / non-finite) gets g0 = ORACLE_GATE_NONE, k = -1.  s0dA is not consulted. */
int oracle_indices(const oracle_config *c, const oracle_sat *s, int64_t n, const float *x,
                   const float *y, const float *z, const float *vx, const float *vy,
                   const float *vz, int32_t *g0, int32_t *k) {
  if (!c || !s || n < 0) return -1;
  double inv_dR, two_over_lambda, cD;
  constants(c, &inv_dR, &two_over_lambda, &cD);
#pragma omp parallel for schedule(static)
  for (int64_t p = 0; p < n; ++p) {
    geom_t g;
    if (geometry(c, s, inv_dR, two_over_lambda, cD, x[p], y[p], z[p], vx[p], vy[p], vz[p], &g)) {
      g0[p] = g.g0;
      k[p] = g.k;
    } else {
      g0[p] = ORACLE_GATE_NONE;
      k[p] = -1;
    }
  }
  return 0;
}

/* Doppler coordinate kf = f_D N / PRF before rounding to a bin (pins of the Doppler readings); NaN for
 * a dropped scatterer. */
int oracle_doppler_coordinate(const oracle_config *c, const oracle_sat *s, int64_t n, const float *x,
                              const float *y, const float *z, const float *vx, const float *vy,
                              const float *vz, double *kf) {
  if (!c || !s || n < 0) return -1;
  double inv_dR, two_over_lambda, cD;
  constants(c, &inv_dR, &two_over_lambda, &cD);
  for (int64_t p = 0; p < n; ++p) {
    geom_t g;
    kf[p] = geometry(c, s, inv_dR, two_over_lambda, cD, x[p], y[p], z[p], vx[p], vy[p], vz[p], &g)
                ? g.kf : NAN;
  }
  return 0;
}

/* O2.  y[g][m] = sum_k T[g][k] exp(+2 pi i ((k m) mod N)/N), m = 0..N-1, NO 1/N (reading A2).
 * T, y: [G][N] complex128. */
int oracle_idft(int32_t G, int32_t N, const double *T, double *y) {
  if (G < 0 || N < 1 || !T || !y) return -1;
  double *w = (double *)malloc((size_t)N * 2 * sizeof(double));
  if (!w) return -2;
  for (int j = 0; j < N; ++j) {
    w[2 * j] = cos(TWO_PI * (double)j / (double)N);
    w[2 * j + 1] = sin(TWO_PI * (double)j / (double)N);
  }
#pragma omp parallel for schedule(static)
  for (int g = 0; g < G; ++g) {
    const double *t = T + (size_t)g * N * 2;
    double *o = y + (size_t)g * N * 2;
    for (int m = 0; m < N; ++m) {
      double sr = 0.0, si = 0.0;
      for (int k = 0; k < N; ++k) {
        const int j = (int)(((int64_t)k * m) % N);
        sr += t[2 * k] * w[2 * j] - t[2 * k + 1] * w[2 * j + 1];
        si += t[2 * k] * w[2 * j + 1] + t[2 * k + 1] * w[2 * j];
      }
      o[2 * m] = sr;
      o[2 * m + 1] = si;
    }
  }
  free(w);
  return 0;
}

/* eq. (1) evaluated at offset |i - x| = d pulses, 0 <= d <= P. */
double oracle_weight(int32_t weight_mode, int32_t P, int64_t d) {
  const double lin = 1.0 - (double)d / (double)P;
  return weight_mode == ORACLE_W_LINEAR ? lin : sqrt(lin);
}

static int64_t pmod(int64_t a, int64_t n) {
  const int64_t r = a % n;
  return r < 0 ? r + n : r;
}

/* O3.  T_all: [n_spectra][G][N] complex128, spectrum u centred on pulse c_u = u P.
 * Y: [n_pulses][G] complex128 for pulses x0 .. x0+n_pulses-1.
 *   Y[x][g] = W_s(x) y_s[g][(x - c_s) mod N] + W_{s+1}(x) y_{s+1}[g][(x - c_{s+1}) mod N],  s = floor(x/P)
 * tail (spectrum s+1 absent): allowed only if final != 0, then Y[x][g] = y_s[g][(x - c_s) mod N].
 * Returns 0, or -3 when a needed spectrum is missing. */
int oracle_synthesize(const oracle_config *c, int32_t n_spectra, const double *T_all, int64_t x0,
                      int64_t n_pulses, int final, double *Y) {
  if (!c || !T_all || !Y || n_pulses < 0 || x0 < 0 || c->pulses_per_update < 1) return -1;
  const int G = c->n_gates, N = c->n_doppler;
  const int64_t P = c->pulses_per_update;
  if (n_pulses == 0) return 0;
  const int64_t s_first = x0 / P, s_last = (x0 + n_pulses - 1) / P;
  if (s_last >= n_spectra) return -3;
  if (s_last + 1 >= n_spectra && !final) return -3;
  const int64_t u_lo = s_first, u_hi = (s_last + 1 < n_spectra) ? s_last + 1 : s_last;
  const size_t grid = (size_t)G * N * 2;
  double *ysig = (double *)malloc((size_t)(u_hi - u_lo + 1) * grid * sizeof(double));
  if (!ysig) return -2;
  for (int64_t u = u_lo; u <= u_hi; ++u) /* step 2 of PAPER.md:99 */
    oracle_idft(G, N, T_all + (size_t)u * grid, ysig + (size_t)(u - u_lo) * grid);
  for (int64_t j = 0; j < n_pulses; ++j) {
    const int64_t x = x0 + j;
    const int64_t s = x / P;
    const int64_t m = x - s * P; /* = x - c_s */
    const double *ys = ysig + (size_t)(s - u_lo) * grid;
    double *out = Y + (size_t)j * G * 2;
    if (s + 1 < n_spectra) {
      const double *yn = ysig + (size_t)(s + 1 - u_lo) * grid;
      const double Ws = oracle_weight(c->weight_mode, (int32_t)P, m);     /* |c_s - x| = m */
      const double Wn = oracle_weight(c->weight_mode, (int32_t)P, P - m); /* |c_{s+1} - x| = P - m */
      const int64_t is = pmod(m, N), in = pmod(m - P, N);
      for (int g = 0; g < G; ++g) { /* steps 3-4 of PAPER.md:100-101 */
        out[2 * g] = Ws * ys[((size_t)g * N + is) * 2] + Wn * yn[((size_t)g * N + in) * 2];
        out[2 * g + 1] = Ws * ys[((size_t)g * N + is) * 2 + 1] + Wn * yn[((size_t)g * N + in) * 2 + 1];
      }
    } else {
      const int64_t is = pmod(m, N);
      for (int g = 0; g < G; ++g) {
        out[2 * g] = ys[((size_t)g * N + is) * 2];
        out[2 * g + 1] = ys[((size_t)g * N + is) * 2 + 1];
      }
    }
  }
  free(ysig);
  return 0;
}

/* REGULAR MODE: "the surface [is] updated at each PRF" and the raw
 * data of a pulse are "obtained by summing the complex contributions from all the facets ... in each range
 * gate".  Point scatterers and satellite in uniform motion from the states given at pulse 0 (reading R5):
 * for pulse j (any sign), t_j = j / PRF, d_j = d + (v_p - v_sat) t_j, R_j = |d_j|, the two-gate linear split
 * (A8) and the complex amplitude of step O1 evaluated at R_j, d_j; no Doppler axis.
 * Y: [n_pulses][G] complex128 for pulses j0 .. j0 + n_pulses - 1; accumulate != 0 adds to Y. */
static void regular_range(const oracle_config *c, const oracle_sat *s, int64_t lo, int64_t hi,
                          const float *x, const float *y, const float *z, const float *vx,
                          const float *vy, const float *vz, const float *s0dA, int64_t j0,
                          int64_t n_pulses, double *Y) {
  double inv_dR, two_over_lambda, cD, b[3];
  constants(c, &inv_dR, &two_over_lambda, &cD);
  unit_boresight(s, b);
  const int G = c->n_gates;
  for (int64_t p = lo; p < hi; ++p) {
    if (!(s0dA[p] > 0.0f)) continue;
    const double dx0 = (double)x[p] - s->pos[0], dy0 = (double)y[p] - s->pos[1], dz0 = (double)z[p] - s->pos[2];
    const double dvx = (double)vx[p] - s->vel[0], dvy = (double)vy[p] - s->vel[1], dvz = (double)vz[p] - s->vel[2];
    const double amp0 = sqrt((double)s0dA[p]);
    for (int64_t jj = 0; jj < n_pulses; ++jj) {
      const double t = (double)(j0 + jj) / c->prf_hz;
      const double dx = fma(dvx, t, dx0), dy = fma(dvy, t, dy0), dz = fma(dvz, t, dz0);
      const double R2 = fma(dz, dz, fma(dy, dy, dx * dx));
      const double R = sqrt(R2);
      const double gf = (R - s->range_gate0_m) * inv_dR;
      if (!(gf >= -1.0 && gf < (double)G)) continue;
      const double g0d = floor(gf);
      const int g0 = (int)g0d;
      const double w1 = gf - g0d, w0 = 1.0 - w1;
      const double q = R * two_over_lambda;
      const double fr = q - floor(q);
      const double cx = dy * b[2] - dz * b[1], cy = dz * b[0] - dx * b[2], cz = dx * b[1] - dy * b[0];
      const double sin2 = (cx * cx + cy * cy + cz * cz) / R2;
      const double A = amp0 * exp(-c->antenna_alpha * sin2) / R2;
      const double re = A * cos(TWO_PI * fr), im = -A * sin(TWO_PI * fr);
      double *row = Y + (size_t)jj * G * 2;
      if (g0 >= 0 && g0 < G) {
        row[2 * g0] += w0 * re;
        row[2 * g0 + 1] += w0 * im;
      }
      if (g0 + 1 >= 0 && g0 + 1 < G) {
        row[2 * (g0 + 1)] += w1 * re;
        row[2 * (g0 + 1) + 1] += w1 * im;
      }
    }
  }
}

int oracle_regular(const oracle_config *c, const oracle_sat *s, int64_t n, const float *x, const float *y,
                   const float *z, const float *vx, const float *vy, const float *vz, const float *s0dA,
                   int64_t j0, int64_t n_pulses, double *Y, int accumulate, int nthreads) {
  if (!c || !s || !Y || n < 0 || n_pulses < 0 || c->n_gates < 1) return -1;
  const int64_t cells = n_pulses * c->n_gates;
  if (!accumulate) memset(Y, 0, (size_t)cells * 2 * sizeof(double));
  if (nthreads <= 1) {
    regular_range(c, s, 0, n, x, y, z, vx, vy, vz, s0dA, j0, n_pulses, Y);
    return 1;
  }
#ifdef _OPENMP
  double *priv = (double *)calloc((size_t)nthreads * (size_t)cells * 2, sizeof(double));
  if (!priv) return -2;
#pragma omp parallel num_threads(nthreads)
  {
    const int t = omp_get_thread_num();
    const int nt = omp_get_num_threads();
    regular_range(c, s, n * t / nt, n * (t + 1) / nt, x, y, z, vx, vy, vz, s0dA, j0, n_pulses,
                  priv + (size_t)t * cells * 2);
  }
  for (int t = 0; t < nthreads; ++t)
    for (int64_t j = 0; j < cells * 2; ++j) Y[j] += priv[(size_t)t * cells * 2 + j];
  free(priv);
  return nthreads;
#else
  regular_range(c, s, 0, n, x, y, z, vx, vy, vz, s0dA, j0, n_pulses, Y);
  return 1;
#endif
}

/* Delay-Doppler burst step: "splitting the data into bursts of 64 pulses,
 * and for each burst performing ... an along-track FFT".  Forward DFT along the pulses of each burst, per gate,
 * written out: Z[b][k][g] = sum_{m<B} Y[b B + m][g] exp(-2 pi i ((k m) mod B)/B), unnormalised, k in natural order.
 * The Doppler-centroid and range-migration corrections of the paper need instrument data and are not part of it.
 * Y: [n_bursts * B][G], Z: [n_bursts][B][G], complex128. */
int oracle_burst_dft(int32_t G, int32_t B, int64_t n_bursts, const double *Y, double *Z) {
  if (G < 1 || B < 1 || n_bursts < 0 || !Y || !Z) return -1;
  double *w = (double *)malloc((size_t)B * 2 * sizeof(double));
  if (!w) return -2;
  for (int j = 0; j < B; ++j) {
    w[2 * j] = cos(TWO_PI * (double)j / (double)B);
    w[2 * j + 1] = -sin(TWO_PI * (double)j / (double)B);
  }
#pragma omp parallel for schedule(static)
  for (int64_t b = 0; b < n_bursts; ++b)
    for (int k = 0; k < B; ++k)
      for (int g = 0; g < G; ++g) {
        double sr = 0.0, si = 0.0;
        for (int m = 0; m < B; ++m) {
          const double *y = Y + (((size_t)b * B + m) * G + g) * 2;
          const int j = (int)(((int64_t)k * m) % B);
          sr += y[0] * w[2 * j] - y[1] * w[2 * j + 1];
          si += y[0] * w[2 * j + 1] + y[1] * w[2 * j];
        }
        double *z = Z + (((size_t)b * B + k) * G + g) * 2;
        z[0] = sr;
        z[1] = si;
      }
  free(w);
  return 0;
}

int oracle_max_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}
