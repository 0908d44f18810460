/*
 * qlp_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, obviously-correct CPU statement of what the QLP GPU transit search computes
 * (arXiv:2302.01293, /root/reference/PAPER.md; readings of every silent/ambiguous point are
 * listed in DESIGN.md "Readings" and SURVEY.md section 8(c)).  IEEE FP64, round-to-nearest,
 * no fused multiply-add (compile with -ffp-contract=off), operations in the order written.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may
 * load this.  It shares no code, header, table or constant generator with the CUDA path under
 * paper_2302_01293_b200/csrc/: every constant below is typed here a second time on purpose.
 *
 * Parity pins (tests/test_oracle_*.py): closed forms, invariants, brute force, library special
 * cases.  The paper prints no spectrum, grid size or S/N value, so "parity unpinned" against
 * paper-printed numbers (only the order of magnitude of the frequency count).
 *
 * Steps (names follow SURVEY.md 8(c)):
 *   O0 constants, cbrt_det      O1 per-star Keplerian grid
 *   O2 prep (Kovacs et al. 2002 weights)
 *   O3 bin index                O4 box scan -> SR(f), best (m, j)
 *   O5 S/N spectrum (footnote 3 at :65)   O6 peaks
 *   O7 per-peak statistics                  O8 trapezoid fit
 *   O9 sigma_w, sigma_r, S/N_pink, detection criteria
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define ORC_PI 0x1.921fb54442d18p+1
/* O0: K_rho = G rho_sun (86400 s/d)^2 = 3 GM_sun / (4 pi R_sun^3) * 86400^2, GM_sun = 1.3271244e20
 * m^3 s^-2, R_sun = 6.957e8 m  ->  702.3999946673047 d^-2 (a literal; never recomputed). */
#define ORC_K_RHO 0x1.5f3333067752fp+9
#define ORC_MAX_WIDTHS 64

typedef struct {
  double samples_per_peak; /* 2.0 */
  double dlogq;            /* 0.1 */
  int32_t noverlap;        /* 3 */
  int32_t uniform_freq;    /* 0; 1 = O1.10c, the comparison grid with equal steps in frequency */
  double qmin_fac;         /* 0.5 */
  double qmax_fac;         /* 2.0 */
  double a_over_rstar_min; /* 2.0 (3.0 for Sectors 59-60) */
  double sector_days;      /* 27.4 PAPER.md:7 */
  /* O1.10, comparison grid only (the earlier search used "an under-sampled frequency grid on the
   * order of 80,000 frequencies or less" and "periods up to only ~56 days").  0 = no cap (the paper's GPU grid). */
  double max_period_days;  /* 0, or e.g. 56.0 */
  int64_t max_freq;        /* 0, or e.g. 80000 */
} orc_config;

typedef struct {
  double t_ref, baseline, p_min, p_max, c_q, u0, h; /* h > 0: f_k = (u0 + k h)^3; h < 0 (O1.10c): f_k = u0 + k (-h) */
  int64_t n_freq;
  int32_t nb_max;
  int32_t status; /* 0 ok; 1: fewer than 2 points; 2: baseline <= 0; 3: f_max <= f_min (or, O1.10c, a frequency
                     step below 1e-9 f_max) */
} orc_star_grid;

typedef struct {
  int64_t k;
  double freq, period, t0, sr, snr, q, depth;
  int32_t m, j, nb, status;
} orc_peak;

/* ---------------------------------------------------------------- O0 */
/* cbrt_det: the DEFINITION of the cube root used by the grid (not an approximation of libm's):
 * frexp, exponent split by 3, eight Newton steps y <- (2y + a/y^2)/3 from y0 = 0.75 + 0.25 a. */
double orc_cbrt_det(double x) {
  int e;
  double mant = frexp(x, &e); /* x = mant * 2^e, mant in [0.5, 1) */
  int q = (e >= 0) ? (e / 3) : -((-e + 2) / 3); /* floor(e / 3) */
  int r = e - 3 * q;                              /* 0, 1, 2 */
  double a = ldexp(mant, r);                      /* [0.5, 4) */
  double y = 0.75 + 0.25 * a;
  for (int it = 0; it < 8; ++it) {
    double y2 = y * y;
    double d = a / y2;
    double s = 2.0 * y;
    double n = s + d;
    y = n / 3.0;
  }
  return ldexp(y, q);
}

/* O1.9: duration ladder in fine bins.  Rungs q_j = qmin_fac (1+dlogq)^j q_circ, j = 0..J-1 with
 * J = floor(ln(qmax_fac/qmin_fac)/ln(1+dlogq)) + 1; in fine bins m_j = floor(noverlap (1+dlogq)^j + 0.5),
 * power by repeated multiplication; duplicates removed.  Defaults -> {3,...,11}.  PAPER.md:19,35. */
int orc_widths(const orc_config* c, int32_t* M) {
  int J = (int)floor(log(c->qmax_fac / c->qmin_fac) / log(1.0 + c->dlogq)) + 1;
  int n = 0;
  double x = 1.0;
  for (int j = 0; j < J; ++j) {
    int m = (int)floor((double)c->noverlap * x + 0.5);
    if (n == 0 || M[n - 1] != m) {
      if (n >= ORC_MAX_WIDTHS) return -1;
      M[n++] = m;
    }
    x = x * (1.0 + c->dlogq);
  }
  return n;
}

/* ---------------------------------------------------------------- O1 */
/* Per-star grid descriptor.  PAPER.md:19 (Keplerian durations, solar density if missing), :23
 * (P_min where a = k R*, P_max = longest continuous stretch or half of it), :35 (samples_per_peak,
 * noverlap).  t strictly increasing, days. */
void orc_grid(const orc_config* c, int64_t n, const double* t, double rho_in, orc_star_grid* g) {
  memset(g, 0, sizeof(*g));
  double rho = (isfinite(rho_in) && rho_in > 0.0) ? rho_in : 1.0; /* O1.1 */
  if (n < 2) { g->status = 1; if (n == 1) g->t_ref = t[0]; return; }
  g->t_ref = t[0];
  double T = t[n - 1] - t[0];
  g->baseline = T;
  /* O1.2: breaks are gaps strictly longer than one sector; L = longest stretch (last - first). */
  int has_break = 0;
  double L = 0.0;
  int64_t first = 0;
  for (int64_t i = 0; i + 1 < n; ++i) {
    if ((t[i + 1] - t[i]) > c->sector_days) {
      double len = t[i] - t[first];
      if (len > L) L = len;
      first = i + 1;
      has_break = 1;
    }
  }
  {
    double len = t[n - 1] - t[first];
    if (len > L) L = len;
  }
  double p_max = has_break ? L : 0.5 * L;
  /* O1.10a: optional period cap of the comparison grid. */
  if (c->max_period_days > 0.0 && p_max > c->max_period_days) p_max = c->max_period_days;
  g->p_max = p_max;
  /* O1.3: Kepler, a/R* = (G rho P^2 / 3 pi)^(1/3)  =>  P_min = sqrt(3 pi k^3 / (K_rho rho)). */
  double D = ORC_K_RHO * rho;
  double k = c->a_over_rstar_min;
  double c3 = (k * k) * k;
  double p_min = sqrt(((3.0 * ORC_PI) * c3) / D);
  g->p_min = p_min;
  /* O1.4: q_circ(f) = (R* / a) / pi = C_q f^(2/3). */
  double c_q = orc_cbrt_det((3.0 * ORC_PI) / D) / ORC_PI;
  g->c_q = c_q;
  if (!(T > 0.0)) { g->status = 2; return; }
  if (!(p_max > 0.0)) { g->status = 3; return; }
  double f_min = 1.0 / p_max;
  double f_max = 1.0 / p_min;
  if (!(f_max > f_min)) { g->status = 3; return; }
  /* O1.6-7: uniform in u = f^(1/3) with step h = qmin_fac C_q / (samples_per_peak T) / 3. */
  double u0 = orc_cbrt_det(f_min);
  double u1 = orc_cbrt_det(f_max);
  double Q = c->qmin_fac * c_q;
  double A = Q / (c->samples_per_peak * T);
  double h = A / 3.0;
  g->n_freq = (int64_t)floor((u1 - u0) / h) + 1;
  /* O1.10b: optional cap on the number of frequencies: the same range in u, under-sampled to exactly max_freq
   * points (step (u1 - u0) / (max_freq - 1)). */
  if (c->max_freq >= 2 && g->n_freq > c->max_freq) {
    h = (u1 - u0) / (double)(c->max_freq - 1);
    g->n_freq = c->max_freq;
  }
  g->u0 = u0;
  g->h = h;
  {
    double u2 = u0 * u0;
    double qlo = Q * u2;
    g->nb_max = (int32_t)ceil(((double)c->noverlap) / qlo);
  }
  /* O1.10c: the comparison grid with equal steps in FREQUENCY (the shape of the earlier CPU search, PAPER.md:13:
   * "an under-sampled frequency grid on the order of 80,000 frequencies or less"): f_k = f_min + k df over the same
   * range [f_min, f_max].  df is the step the f^(1/3) law has at f_min, where it is finest (d(u^3)/dk = 3 u^2 h =
   * A u0^2), so that no part of the range is sampled more coarsely than the GPU grid samples it; when that takes
   * more than max_freq points the range is under-sampled to exactly max_freq of them.  nb_k keeps the Keplerian
   * law of O1.8 at f_k.  The descriptor holds u0 = f_min and h = -df: the sign of h marks the grid's kind.
   * A step below 1e-9 f_max is refused (status 3): cbrt_det is accurate to a few 1e-16, so above that bound
   * u_k = cbrt_det(f_k) and with it nb_k are monotone in k. */
  if (c->uniform_freq) {
    double df = A * (u0 * u0);
    g->n_freq = (int64_t)floor((f_max - f_min) / df) + 1;
    if (c->max_freq >= 2 && g->n_freq > c->max_freq) {
      df = (f_max - f_min) / (double)(c->max_freq - 1);
      g->n_freq = c->max_freq;
    }
    if (!(df > 1e-9 * f_max)) { g->status = 3; g->n_freq = 0; g->nb_max = 0; g->u0 = 0.0; g->h = 0.0; return; }
    g->u0 = f_min;
    g->h = -df;
  }
}

/* O1.8: frequency k and its number of fine phase bins. */
void orc_freq(const orc_config* c, const orc_star_grid* g, int64_t k, double* f, int32_t* nb) {
  double Q = c->qmin_fac * g->c_q;
  if (g->h < 0.0) { /* O1.10c: equal steps in frequency, Keplerian nb at f_k */
    double fk = g->u0 + ((double)k) * (-g->h);
    double u = orc_cbrt_det(fk);
    double u2 = u * u;
    *f = fk;
    double qlo = Q * u2;
    *nb = (int32_t)ceil(((double)c->noverlap) / qlo);
    return;
  }
  double u = g->u0 + ((double)k) * g->h;
  double u2 = u * u;
  *f = u2 * u;
  double qlo = Q * u2;
  *nb = (int32_t)ceil(((double)c->noverlap) / qlo);
}

void orc_freqs(const orc_config* c, const orc_star_grid* g, int64_t k0, int64_t k1, double* f, int32_t* nb) {
  for (int64_t k = k0; k < k1; ++k) orc_freq(c, g, k, &f[k - k0], &nb[k - k0]);
}

/* ---------------------------------------------------------------- O2 */
/* Kovacs et al. (2002) weighting: w_i = dy_i^-2 / sum dy^-2, weighted-mean-subtracted series. */
void orc_prep(int64_t n, const double* t, const double* y, const double* dy, double t_ref,
              double* tau, double* w, double* wy) {
  double W = 0.0;
  for (int64_t i = 0; i < n; ++i) W += 1.0 / (dy[i] * dy[i]);
  double ybar = 0.0;
  for (int64_t i = 0; i < n; ++i) {
    w[i] = (1.0 / (dy[i] * dy[i])) / W;
    ybar += w[i] * y[i];
  }
  for (int64_t i = 0; i < n; ++i) {
    double yt = y[i] - ybar;
    wy[i] = w[i] * yt;
    tau[i] = t[i] - t_ref;
  }
}

/* ---------------------------------------------------------------- O3 */
/* Bin index of one point at one frequency; what the CUDA path must reproduce bit for bit.
 * Reading A17: p = fl64(f * tau) is the one rounded operation; the bin is then
 *   b = floor( nb * (p - floor(p)) )   evaluated EXACTLY (no second rounding, hence b <= nb-1
 * always and no clamp).  p - floor(p) is exact in FP64; its product with the integer nb needs up to
 * 53 + 15 bits, so it is formed in 128-bit integer arithmetic: ph = M * 2^-sh with M a 53-bit
 * integer, b = (M * nb) >> sh.  Requires 0 <= p < 2^52 (tau >= 0, f > 0). */
static inline int32_t orc_bin1(double f, int32_t nb, double tau) {
  double p = f * tau;
  double c = floor(p);
  double ph = p - c;                 /* exact, in [0, 1) */
  if (ph <= 0.0) return 0;
  int e;
  double mant = frexp(ph, &e);       /* ph = mant * 2^e, mant in [0.5, 1), e <= 0 */
  uint64_t M = (uint64_t)ldexp(mant, 53);          /* integer, < 2^53 */
  int sh = 53 - e;                   /* ph = M * 2^-sh, sh >= 53 */
  unsigned __int128 prod = (unsigned __int128)M * (unsigned __int128)(uint32_t)nb;
  if (sh >= 128) return 0;
  return (int32_t)(uint64_t)(prod >> sh);
}

void orc_bins(double f, int32_t nb, int64_t n, const double* tau, int32_t* b) {
  for (int64_t i = 0; i < n; ++i) b[i] = orc_bin1(f, nb, tau[i]);
}

/* ---------------------------------------------------------------- O3+O4 */
/* One frequency: fold into nb bins, then try every start bin j and every width m in M (wrapped).
 * SR = max s^2 / (r (1 - r)); ties -> smaller m, then smaller j; all-zero -> SR 0, (M[0], 0).
 * Hw/Hs are caller scratch of nb doubles.  r_best/s_best may be NULL. */
void orc_sr_one(int64_t n, const double* tau, const double* w, const double* wy, double f, int32_t nb,
                int nM, const int32_t* M, double* Hw, double* Hs,
                double* sr, int32_t* m_best, int32_t* j_best, double* r_best, double* s_best) {
  for (int32_t b = 0; b < nb; ++b) { Hw[b] = 0.0; Hs[b] = 0.0; }
  for (int64_t i = 0; i < n; ++i) {
    int32_t b = orc_bin1(f, nb, tau[i]);
    Hw[b] += w[i];
    Hs[b] += wy[i];
  }
  double best = 0.0, rb = 0.0, sb = 0.0;
  int32_t mb = M[0], jb = 0;
  for (int im = 0; im < nM; ++im) {   /* widths ascending: first strict improvement wins ties */
    int32_t m = M[im];
    for (int32_t j = 0; j < nb; ++j) {
      double r = 0.0, s = 0.0;
      for (int32_t l = 0; l < m; ++l) {
        int32_t b = j + l;
        if (b >= nb) b -= nb;
        r += Hw[b];
        s += Hs[b];
      }
      double val = (r > 0.0 && r < 1.0) ? (s * s) / (r * (1.0 - r)) : 0.0;
      if (val > best) { best = val; mb = m; jb = j; rb = r; sb = s; }
    }
  }
  *sr = best; *m_best = mb; *j_best = jb;
  if (r_best) *r_best = rb;
  if (s_best) *s_best = sb;
}

/* Whole spectrum of one star over its own grid. Outputs have g->n_freq entries. */
int orc_spectrum_star(const orc_config* c, const orc_star_grid* g, int64_t n, const double* t,
                      const double* y, const double* dy, double* sr, int32_t* m_best, int32_t* j_best) {
  if (g->status != 0 || g->n_freq <= 0) return 0;
  int32_t M[ORC_MAX_WIDTHS];
  int nM = orc_widths(c, M);
  if (nM <= 0) return -1;
  double* tau = (double*)malloc(sizeof(double) * (size_t)n * 3);
  double* Hw = (double*)malloc(sizeof(double) * (size_t)g->nb_max * 2);
  if (!tau || !Hw) { free(tau); free(Hw); return -2; }
  double* w = tau + n;
  double* wy = w + n;
  double* Hs = Hw + g->nb_max;
  orc_prep(n, t, y, dy, g->t_ref, tau, w, wy);
  for (int64_t k = 0; k < g->n_freq; ++k) {
    double f; int32_t nb;
    orc_freq(c, g, k, &f, &nb);
    orc_sr_one(n, tau, w, wy, f, nb, nM, M, Hw, Hs, &sr[k], &m_best[k], &j_best[k], NULL, NULL);
  }
  free(tau); free(Hw);
  return 0;
}

/* Test helpers (no new arithmetic: they only call orc_prep / orc_freq / orc_sr_one / orc_bin1 above).
 * orc_spectrum_samples: O3+O4 of one star at the selected grid indices ks[0..nk), OpenMP over the samples, so that
 * long-baseline stars (10^5..10^6 frequencies) can be checked on a sample.  r_best/s_best optional (NULL). */
int orc_spectrum_samples(const orc_config* c, const orc_star_grid* g, int64_t n, const double* t, const double* y,
                         const double* dy, int64_t nk, const int64_t* ks, double* sr, int32_t* m_best,
                         int32_t* j_best) {
  if (g->status != 0 || g->n_freq <= 0 || nk <= 0) return 0;
  int32_t M[ORC_MAX_WIDTHS];
  int nM = orc_widths(c, M);
  if (nM <= 0) return -1;
  double* tau = (double*)malloc(sizeof(double) * (size_t)(n > 0 ? n : 1) * 3);
  if (!tau) return -2;
  double* w = tau + n;
  double* wy = w + n;
  orc_prep(n, t, y, dy, g->t_ref, tau, w, wy);
  int err = 0;
#pragma omp parallel
  {
    double* Hw = (double*)malloc(sizeof(double) * (size_t)g->nb_max * 2);
    if (!Hw) err = -2;
#pragma omp for schedule(dynamic, 1)
    for (int64_t i = 0; i < nk; ++i) {
      if (!Hw || ks[i] < 0 || ks[i] >= g->n_freq) { if (Hw) err = -3; continue; }
      double f; int32_t nb;
      orc_freq(c, g, ks[i], &f, &nb);
      orc_sr_one(n, tau, w, wy, f, nb, nM, M, Hw, Hw + g->nb_max, &sr[i], &m_best[i], &j_best[i], NULL, NULL);
    }
    free(Hw);
  }
  free(tau);
  return err;
}

/* orc_box_values: the value s^2 / (r (1 - r)) (0 outside 0 < r < 1) of GIVEN boxes (ms[i] bins from start bin
 * js[i], wrapped) at grid indices ks[i] of one star: lets a test check that a box reported by another
 * implementation is as good as the oracle's best one.  Sums run over the points in time order. */
int orc_box_values(const orc_config* c, const orc_star_grid* g, int64_t n, const double* t, const double* y,
                   const double* dy, int64_t nk, const int64_t* ks, const int32_t* ms, const int32_t* js,
                   double* val) {
  if (g->status != 0 || g->n_freq <= 0 || nk <= 0) return 0;
  double* tau = (double*)malloc(sizeof(double) * (size_t)(n > 0 ? n : 1) * 3);
  if (!tau) return -2;
  double* w = tau + n;
  double* wy = w + n;
  orc_prep(n, t, y, dy, g->t_ref, tau, w, wy);
#pragma omp parallel for schedule(dynamic, 4)
  for (int64_t i = 0; i < nk; ++i) {
    double f; int32_t nb;
    orc_freq(c, g, ks[i], &f, &nb);
    double r = 0.0, s = 0.0;
    for (int64_t p = 0; p < n; ++p) {
      int32_t d = orc_bin1(f, nb, tau[p]) - js[i];
      if (d < 0) d += nb;
      if (d < ms[i]) { r += w[p]; s += wy[p]; }
    }
    val[i] = (r > 0.0 && r < 1.0) ? (s * s) / (r * (1.0 - r)) : 0.0;
  }
  free(tau);
  return 0;
}

/* ---------------------------------------------------------------- O5 */
static int cmp_double(const void* a, const void* b) {
  double x = *(const double*)a, y = *(const double*)b;
  return (x > y) - (x < y);
}
static double median_sorted(const double* v, int64_t n) {
  return (n & 1) ? v[n / 2] : 0.5 * (v[n / 2 - 1] + v[n / 2]);
}

/* Sturges' law, PAPER.md:65 footnote 3: N = 1 + 3.322 log10(n), rounded to the nearest integer. */
int32_t orc_sturges(int64_t n) {
  int32_t N = (int32_t)floor(1.0 + 3.322 * log10((double)n) + 0.5);
  return N < 1 ? 1 : N;
}

/* S/N(f) = (SR - trend)/sigma: trend = linear interpolation through the medians
 * of N equal-width frequency bins (bin centres; constant outside); sigma = 1.4826 MAD(SR).
 * trend/sigma outputs optional (NULL). */
void orc_snr(int64_t n, const double* f, const double* sr, double* snr, double* trend_out, double* sigma_out) {
  if (n <= 0) return;
  int32_t N = orc_sturges(n);
  double f0 = f[0];
  double span = f[n - 1] - f0;
  double* sorted = (double*)malloc(sizeof(double) * (size_t)n);
  int32_t* bin = (int32_t*)malloc(sizeof(int32_t) * (size_t)n);
  double* cx = (double*)malloc(sizeof(double) * (size_t)N * 2);
  double* cy = cx + N;
  int64_t* cnt = (int64_t*)calloc((size_t)N, sizeof(int64_t));
  for (int64_t k = 0; k < n; ++k) {
    int32_t b = 0;
    if (span > 0.0) {
      b = (int32_t)(((f[k] - f0) / span) * (double)N);
      if (b > N - 1) b = N - 1;
    }
    bin[k] = b;
    cnt[b]++;
  }
  int32_t nk = 0;
  for (int32_t b = 0; b < N; ++b) {
    if (cnt[b] == 0) continue;  /* empty bins are dropped */
    int64_t c = 0;
    for (int64_t k = 0; k < n; ++k) if (bin[k] == b) sorted[c++] = sr[k];
    qsort(sorted, (size_t)c, sizeof(double), cmp_double);
    cx[nk] = f0 + (((double)b + 0.5) * span) / (double)N;
    cy[nk] = median_sorted(sorted, c);
    nk++;
  }
  /* sigma = 1.4826 * median |SR - median(SR)| (raw spectrum; reading A21). */
  memcpy(sorted, sr, sizeof(double) * (size_t)n);
  qsort(sorted, (size_t)n, sizeof(double), cmp_double);
  double med = median_sorted(sorted, n);
  for (int64_t k = 0; k < n; ++k) sorted[k] = fabs(sr[k] - med);
  qsort(sorted, (size_t)n, sizeof(double), cmp_double);
  double sigma = 1.4826 * median_sorted(sorted, n);
  if (sigma_out) *sigma_out = sigma;
  int32_t seg = 0;
  for (int64_t k = 0; k < n; ++k) {
    double x = f[k], tr;
    if (x <= cx[0]) tr = cy[0];
    else if (x >= cx[nk - 1]) tr = cy[nk - 1];
    else {
      while (seg + 1 < nk - 1 && x >= cx[seg + 1]) seg++;
      while (seg > 0 && x < cx[seg]) seg--;
      double slope = (cy[seg + 1] - cy[seg]) / (cx[seg + 1] - cx[seg]);
      tr = slope * (x - cx[seg]) + cy[seg];
    }
    if (trend_out) trend_out[k] = tr;
    snr[k] = (sigma > 0.0) ? (sr[k] - tr) / sigma : 0.0;
  }
  free(sorted); free(bin); free(cx); free(cnt);
}

/* ---------------------------------------------------------------- O6 */
/* Rank 1 = argmax S/N (ties -> lower k).  Ranks 2..K = remaining strict local maxima
 * (snr[k] > snr[k-1] and snr[k] >= snr[k+1]; ends compare with their one neighbour) by descending
 * S/N, ties -> lower k.  Returns the number of peaks written (<= K). */
int orc_peak_indices(int64_t n, const double* snr, int K, int64_t* out) {
  if (n <= 0 || K <= 0) return 0;
  int64_t k1 = 0;
  for (int64_t k = 1; k < n; ++k) if (snr[k] > snr[k1]) k1 = k;
  int cnt = 0;
  out[cnt++] = k1;
  while (cnt < K) {
    int64_t best = -1;
    for (int64_t k = 0; k < n; ++k) {
      int lm = (k == 0 || snr[k] > snr[k - 1]) && (k == n - 1 || snr[k] >= snr[k + 1]);
      if (n == 1) lm = 0;
      if (!lm) continue;
      int used = 0;
      for (int i = 0; i < cnt; ++i) if (out[i] == k) used = 1;
      if (used) continue;
      /* descending order: must not exceed the previous pick (ties resolved by index) */
      if (best < 0 || snr[k] > snr[best]) best = k;
    }
    if (best < 0) break;
    out[cnt++] = best;
  }
  return cnt;
}

/* Peak record at frequency k: refold to get (r, s) at the best window; q = m/nb; depth
 * delta = -s / (r (1 - r)) (positive for a dip); T0 = t_ref + ((j + m/2)/nb)/f.  PAPER.md:44. */
void orc_peak_record(const orc_config* c, const orc_star_grid* g, int64_t n, const double* t, const double* y,
                     const double* dy, int64_t k, double snr_k, orc_peak* p) {
  int32_t M[ORC_MAX_WIDTHS];
  int nM = orc_widths(c, M);
  double* tau = (double*)malloc(sizeof(double) * (size_t)n * 3);
  double* w = tau + n;
  double* wy = w + n;
  orc_prep(n, t, y, dy, g->t_ref, tau, w, wy);
  double f; int32_t nb;
  orc_freq(c, g, k, &f, &nb);
  double* Hw = (double*)malloc(sizeof(double) * (size_t)nb * 2);
  double sr, r, s; int32_t m, j;
  orc_sr_one(n, tau, w, wy, f, nb, nM, M, Hw, Hw + nb, &sr, &m, &j, &r, &s);
  p->k = k; p->freq = f; p->period = 1.0 / f; p->sr = sr; p->snr = snr_k;
  p->m = m; p->j = j; p->nb = nb; p->status = 0;
  p->q = (double)m / (double)nb;
  p->depth = (r > 0.0 && r < 1.0) ? -s / (r * (1.0 - r)) : 0.0;
  p->t0 = g->t_ref + (((double)j + 0.5 * (double)m) / (double)nb) / f;
  free(tau); free(Hw);
}

/* ---------------------------------------------------------------- batch driver */
/* Whole path for a CSR batch, OpenMP over stars only.  sr/m/j/snr are [total_freq] with freq_ptr
 * offsets (computed by the caller from orc_grid); snr may be NULL; peaks [S*K] may be NULL. */
int orc_batch(const orc_config* c, int64_t S, const int64_t* row_ptr, const double* t, const double* y,
              const double* dy, const double* rho, const orc_star_grid* grids, const int64_t* freq_ptr,
              double* sr, int32_t* mb, int32_t* jb, double* snr, int K, orc_peak* peaks) {
  int err = 0;
#pragma omp parallel for schedule(dynamic, 1)
  for (int64_t s = 0; s < S; ++s) {
    const orc_star_grid* g = &grids[s];
    int64_t a = row_ptr[s], n = row_ptr[s + 1] - row_ptr[s];
    int64_t fo = freq_ptr[s], nf = freq_ptr[s + 1] - freq_ptr[s];
    if (peaks) for (int i = 0; i < K; ++i) { memset(&peaks[s * K + i], 0, sizeof(orc_peak)); peaks[s * K + i].k = -1; peaks[s * K + i].status = 1; }
    if (g->status != 0 || nf <= 0) continue;
    int rc = orc_spectrum_star(c, g, n, t + a, y + a, dy + a, sr + fo, mb + fo, jb + fo);
    if (rc != 0) { err = rc; continue; }
    if (!snr && !peaks) continue;
    double* f = (double*)malloc(sizeof(double) * (size_t)nf);
    int32_t* nbv = (int32_t*)malloc(sizeof(int32_t) * (size_t)nf);
    double* sn = snr ? snr + fo : (double*)malloc(sizeof(double) * (size_t)nf);
    orc_freqs(c, g, 0, nf, f, nbv);
    orc_snr(nf, f, sr + fo, sn, NULL, NULL);
    if (peaks) {
      int64_t idx[64];
      int kk = K > 64 ? 64 : K;
      int np = orc_peak_indices(nf, sn, kk, idx);
      for (int i = 0; i < np; ++i) orc_peak_record(c, g, n, t + a, y + a, dy + a, idx[i], sn[idx[i]], &peaks[s * K + i]);
    }
    if (!snr) free(sn);
    free(f); free(nbv);
  }
  (void)rho;
  return err;
}

int orc_sizeof_grid(void) { return (int)sizeof(orc_star_grid); }
int orc_sizeof_peak(void) { return (int)sizeof(orc_peak); }
int orc_sizeof_config(void) { return (int)sizeof(orc_config); }

/* ---------------------------------------------------------------- O7 */
/* "Other statistics" of a peak: "the number of points in, before, and after transit, number of
 * transits, and out-of-transit magnitude level.  In order for a transit to count toward the number of
 * transits, we require there to be data within 0.5 transit durations of the expected mid-transit time."
 * Readings (O7): P = 1/f, duration D = q P with q = m/nb from the BLS; for every point
 *   x = (t - T0)/P;  n = floor(x + 0.5);  dt = (x - n) P            (time from the nearest mid-transit)
 *   in transit   : |dt| <= D/2            (this is also "data within 0.5 durations of the mid-time")
 *   before/after : one duration wide, adjacent to the transit: -1.5 D <= dt < -D/2,  D/2 < dt <= 1.5 D
 *   n_transits   : number of distinct n that own at least one in-transit point
 *   oot level    : weighted mean (weights dy^-2) of y over the points that are not in transit.
 * FP64, no FMA, operations in the order written (the classification is an integer decision). */
typedef struct {
  int32_t n_in, n_before, n_after, n_transits;
  double oot_level, duration;
} orc_peak_stats;

void orc_peak_statistics(int64_t n, const double* t, const double* y, const double* dy, double f, int32_t m,
                         int32_t nb, double t0, orc_peak_stats* out) {
  double P = 1.0 / f;
  double q = (double)m / (double)nb;
  double D = q * P;
  double hD = 0.5 * D, wD = 1.5 * D;
  int32_t n_in = 0, n_before = 0, n_after = 0, n_tr = 0;
  double sw = 0.0, swy = 0.0;
  int have_prev = 0;
  double prev_n = 0.0;
  for (int64_t i = 0; i < n; ++i) {
    double x = (t[i] - t0) / P;
    double cyc = floor(x + 0.5);
    double dt = (x - cyc) * P;
    int in = fabs(dt) <= hD;
    if (in) {
      ++n_in;
      if (!have_prev || cyc != prev_n) ++n_tr;  /* t is increasing: in-transit points of one cycle are adjacent */
      have_prev = 1; prev_n = cyc;
    } else {
      double w = 1.0 / (dy[i] * dy[i]);
      sw += w; swy += w * y[i];
      if (dt < -hD && dt >= -wD) ++n_before;
      if (dt > hD && dt <= wD) ++n_after;
    }
  }
  out->n_in = n_in; out->n_before = n_before; out->n_after = n_after; out->n_transits = n_tr;
  out->oot_level = (sw > 0.0) ? swy / sw : 0.0;
  out->duration = D;
}
int orc_sizeof_peak_stats(void) { return (int)sizeof(orc_peak_stats); }

/* ---------------------------------------------------------------- O8 */
/* Trapezoid model fit of one peak: "a trapezoid model parameterized by the orbital period (P),
 * transit epoch (T0), depth (delta), duration divided by orbital period (q), duration of ingress divided by
 * transit duration (q_in), and out-of-transit magnitude level (z).  P is fixed to the BLS period while other
 * parameters are fit using initial guesses from BLS.  To speed up the fit, we only fit data within two transit
 * durations of the transit center.  We place bounds on q between 0 and 1, and q_in between 0 (perfectly
 * box-shaped) and 0.5 (V-shaped)."  The paper names no optimiser; readings (O8):
 *   data     : P = 1/f, q0 = m/nb, D0 = q0 P; x = (t - T0_bls)/P; n = floor(x + 0.5); dt = (x - n) P (as O7);
 *              the points with |dt| <= 2 D0 are the data of the fit, fixed for the whole fit; w = dy^-2.
 *   model    : y ~ z - delta * sh(|dt - c|), c = T0 - T0_bls, D = q P, half = D/2, ing = q_in D,
 *              sh(u) = 0 for u >= half, (half - u)/ing for half - u < ing, else 1   (delta > 0 is a dip, as O6).
 *   linear   : for given (c, q, q_in), z and delta are the weighted least-squares solution (they enter
 *              linearly); chi2 = sum w (y - model)^2 with that solution.  If the weighted variance of sh is
 *              below 1e-9 (no point, or every point, at one level) delta = 0, z = weighted mean.
 *   search   : compass search over (c, q, q_in) from (0, q0, 0.25) with steps (D0/4, q0/4, 0.125), bounds
 *              c in [-D0, D0], q in [0, 1], q_in in [0, 0.5].  One sweep evaluates chi2 at the (up to) six
 *              neighbours theta +- h_d e_d (order c+, c-, q+, q-, q_in+, q_in-; clipped to the bounds, skipped
 *              if the clipped value is the current one), takes the FIRST neighbour in that order whose chi2 is
 *              within tol of the smallest of them, and moves there iff it lowers chi2 by more than tol; a sweep
 *              that does not move halves the steps; 24 halvings; no sweep starts once 600 evaluations are
 *              spent (so at most 605).  tol = max(1e-9 chi2_best, 1e-12 G), chi2_best the current value and
 *              G = sum w (y - ybar)^2 over the window.  chi2 values of two implementations differ by ~1e-15 G
 *              (FP64 sums of ~10^3..10^5 terms in different orders), a million times less than tol on real data
 *              (chi2 ~ G), so neither the choice of the neighbour nor the acceptance depends on the order in
 *              which the points are added up -- except when a difference lands within that noise of tol itself,
 *              about once in 10^6 fits (once in 10^3 on noise-free data, where chi2 -> 0 and the 1e-12 G floor
 *              is what stops the search).  (Reading changed in round 2: the first rule, "try the six moves in
 *              turn, accept iff chi2 strictly decreases", was decided by rounding noise wherever chi2 is flat;
 *              PAPER.md:44 names no optimiser.)
 * FP64; the sums run over the selected points in time order. */
typedef struct {
  double t0, depth, q, q_in, z, chi2, chi2_init;
  int32_t n_fit, n_eval, status, pad_;
} orc_trapezoid;

typedef struct { int64_t n; const double *dt, *yt, *w; double A, ybar, G, P; } orc_fit_data;

static double orc_trap_shape(double u, double half, double ing) {
  if (u >= half) return 0.0;
  double d = half - u;
  if (d < ing) return d / ing;
  return 1.0;
}

/* chi2 at (c, q, q_in); also the linear solution (delta, z). */
static double orc_trap_chi2(const orc_fit_data* fd, double c, double q, double qin, double* delta, double* z) {
  double D = q * fd->P, half = 0.5 * D, ing = qin * D;
  double B = 0.0, Cc = 0.0, F = 0.0;
  for (int64_t i = 0; i < fd->n; ++i) {
    double sh = orc_trap_shape(fabs(fd->dt[i] - c), half, ing);
    double wsh = fd->w[i] * sh;
    B += wsh; Cc += wsh * sh; F += wsh * fd->yt[i];
  }
  double V = Cc - B * B / fd->A;          /* A times the weighted variance of sh */
  double dl = 0.0;
  if (V > 1e-9 * fd->A) dl = -F / V;      /* yt is centred: sum w yt = 0 */
  double zc = dl * B / fd->A;             /* z - ybar */
  double chi2 = 0.0;
  for (int64_t i = 0; i < fd->n; ++i) {
    double sh = orc_trap_shape(fabs(fd->dt[i] - c), half, ing);
    double r = fd->yt[i] - zc + dl * sh;
    chi2 += fd->w[i] * r * r;
  }
  *delta = dl; *z = fd->ybar + zc;
  return chi2;
}

/* The data of a fit (window selection, weights, centring).  Returns n_fit; buf holds 3 n doubles. */
static int64_t orc_fit_select(int64_t n, const double* t, const double* y, const double* dy, double P, double D0,
                              double t0_bls, double* buf, orc_fit_data* fd) {
  double win = 2.0 * D0;
  double *dtv = buf, *yv = buf + n, *wv = buf + 2 * n;
  int64_t nf = 0;
  for (int64_t i = 0; i < n; ++i) {
    double x = (t[i] - t0_bls) / P;
    double cyc = floor(x + 0.5);
    double dt = (x - cyc) * P;
    if (fabs(dt) <= win) { dtv[nf] = dt; yv[nf] = y[i]; wv[nf] = 1.0 / (dy[i] * dy[i]); ++nf; }
  }
  double A = 0.0, E = 0.0, G = 0.0;
  for (int64_t i = 0; i < nf; ++i) { A += wv[i]; E += wv[i] * yv[i]; }
  double ybar = nf > 0 ? E / A : 0.0;
  for (int64_t i = 0; i < nf; ++i) { yv[i] = yv[i] - ybar; G += wv[i] * yv[i] * yv[i]; }
  fd->n = nf; fd->dt = dtv; fd->yt = yv; fd->w = wv; fd->A = A; fd->ybar = ybar; fd->G = G; fd->P = P;
  return nf;
}

void orc_trapezoid_fit(int64_t n, const double* t, const double* y, const double* dy, double f, int32_t m,
                       int32_t nb, double t0_bls, orc_trapezoid* out) {
  memset(out, 0, sizeof(*out));
  double P = 1.0 / f;
  double q0 = (double)m / (double)nb;
  double D0 = q0 * P;
  double* buf = (double*)malloc(sizeof(double) * (size_t)(n > 0 ? n : 1) * 3);
  orc_fit_data fd;
  int64_t nf = orc_fit_select(n, t, y, dy, P, D0, t0_bls, buf, &fd);
  out->n_fit = (int32_t)nf;
  out->t0 = t0_bls; out->q = q0; out->q_in = 0.25;
  if (nf < 5) { out->status = 2; free(buf); return; }
  double th[3] = {0.0, q0, 0.25};
  double h[3] = {0.25 * D0, 0.25 * q0, 0.125};
  const double lo[3] = {-D0, 0.0, 0.0}, hi[3] = {D0, 1.0, 0.5};
  double dl, z;
  double best = orc_trap_chi2(&fd, th[0], th[1], th[2], &dl, &z);
  int n_eval = 1;
  out->chi2_init = best;
  const double tol_floor = 1e-12 * fd.G;
  for (int level = 0; level < 24 && n_eval < 600; ++level) {
    int moved = 1;
    while (moved && n_eval < 600) {
      moved = 0;
      double tol = 1e-9 * best;
      if (tol < tol_floor) tol = tol_floor;
      double chi[6], dlk[6], zk[6], vk[6];
      int have[6];
      double cmin = 0.0;
      int any = 0;
      for (int k = 0; k < 6; ++k) {          /* k = 2 d + sg: c+, c-, q+, q-, q_in+, q_in- */
        int d = k >> 1, sg = k & 1;
        double c[3] = {th[0], th[1], th[2]};
        double v = sg == 0 ? th[d] + h[d] : th[d] - h[d];
        if (v < lo[d]) v = lo[d];
        if (v > hi[d]) v = hi[d];
        have[k] = (v != th[d]);
        if (!have[k]) continue;
        c[d] = v; vk[k] = v;
        chi[k] = orc_trap_chi2(&fd, c[0], c[1], c[2], &dlk[k], &zk[k]);
        ++n_eval;
        if (!any || chi[k] < cmin) cmin = chi[k];
        any = 1;
      }
      if (!any) break;
      int sel = -1;
      for (int k = 0; k < 6 && sel < 0; ++k) if (have[k] && chi[k] <= cmin + tol) sel = k;
      if (chi[sel] < best - tol) { best = chi[sel]; th[sel >> 1] = vk[sel]; dl = dlk[sel]; z = zk[sel]; moved = 1; }
    }
    h[0] *= 0.5; h[1] *= 0.5; h[2] *= 0.5;
  }
  out->t0 = t0_bls + th[0]; out->q = th[1]; out->q_in = th[2];
  out->depth = dl; out->z = z; out->chi2 = best; out->n_eval = n_eval; out->status = 0;
  free(buf);
}
/* chi2 (and the linear solution) of the same data at given (c, q, q_in): lets a test check a fit found elsewhere.
 * res = {chi2, depth, z}; returns n_fit. */
int64_t orc_trapezoid_chi2_at(int64_t n, const double* t, const double* y, const double* dy, double f, int32_t m,
                              int32_t nb, double t0_bls, double c, double q, double qin, double* res) {
  double P = 1.0 / f;
  double D0 = (double)m / (double)nb * P;
  double* buf = (double*)malloc(sizeof(double) * (size_t)(n > 0 ? n : 1) * 3);
  orc_fit_data fd;
  int64_t nf = orc_fit_select(n, t, y, dy, P, D0, t0_bls, buf, &fd);
  res[0] = res[1] = res[2] = 0.0;
  if (nf > 0) res[0] = orc_trap_chi2(&fd, c, q, qin, &res[1], &res[2]);
  free(buf);
  return nf;
}
int orc_sizeof_trapezoid(void) { return (int)sizeof(orc_trapezoid); }

/* ---------------------------------------------------------------- O9 */
/* Noise estimates, signal-to-pink-noise and the detection criteria, PAPER.md:45-51, :55:
 *   "we subtract the trapezoid model from the light curve and estimate the white noise (sigma_w) and red noise
 *    (sigma_r) on the timescale of the transit duration" ... Eq. 2:
 *        S/N_pink = delta / sqrt(sigma_w^2 / n_t + sigma_r^2 / N_t),
 *    n_t the number of points in transit, N_t the number of transits ... "replacing delta with the integral over
 *    the full trapezoid model" ... "detection criteria of at least two transits, S/N_pink > 9, and ... S/N > 9".
 * The VARTOOLS noise recipe is not in the paper; readings (O9, after Pont et al. 2006):
 *   residual r_i = y_i - (z - delta sh_i) over ALL points of the star, sh as in O8 with the fitted T0, q, q_in;
 *   sigma_w^2 = mean (r - mean r)^2 (unweighted);
 *   time bins of one transit duration D = q P counted from the first point, b_i = floor((t_i - t_first)/D);
 *   m_b, n_b = mean and count of every non-empty bin;  sigma_bin^2 = mean_b (m_b - mean_b m)^2;
 *   sigma_r^2 = max(0, sigma_bin^2 - sigma_w^2 mean_b(1/n_b))   (the white part of the binned scatter removed);
 *   n_t, N_t as in O7 (|dt| <= D/2; a transit counts if it owns an in-transit point) with the fitted T0 and D;
 *   delta_eff = delta (1 - q_in)   (the integral of the unit trapezoid over the duration, divided by D);
 *   S/N_pink = delta_eff / sqrt(sigma_w^2/n_t + sigma_r^2/N_t), 0 if n_t = 0 or the denominator is 0;
 *   detected = N_t >= 2 and S/N_pink > 9 and S/N > 9. */
typedef struct {
  double sigma_w, sigma_r, depth_eff, snr_pink;
  int32_t n_t, n_transits, n_bins, detected;
} orc_pink;

void orc_pink_noise(int64_t n, const double* t, const double* y, double f, double T0, double delta, double q,
                    double qin, double z, double snr, orc_pink* out) {
  memset(out, 0, sizeof(*out));
  if (n <= 0) return;
  double P = 1.0 / f;
  double D = q * P, half = 0.5 * D, ing = qin * D;
  double* r = (double*)malloc(sizeof(double) * (size_t)n);
  int32_t n_t = 0, n_tr = 0;
  int have_prev = 0;
  double prev_cyc = 0.0, sum = 0.0;
  for (int64_t i = 0; i < n; ++i) {
    double x = (t[i] - T0) / P;
    double cyc = floor(x + 0.5);
    double dt = (x - cyc) * P;
    double u = fabs(dt);
    r[i] = y[i] - (z - delta * orc_trap_shape(u, half, ing));
    sum += r[i];
    if (u <= half) {
      ++n_t;
      if (!have_prev || cyc != prev_cyc) ++n_tr;
      have_prev = 1; prev_cyc = cyc;
    }
  }
  double rbar = sum / (double)n, ss = 0.0;
  for (int64_t i = 0; i < n; ++i) ss += (r[i] - rbar) * (r[i] - rbar);
  double var_w = ss / (double)n;
  /* bins of one duration; t increases, so a bin is a run of consecutive points */
  double var_bin = 0.0, mean_inv = 0.0;
  int32_t nbins = 0;
  if (D > 0.0) {
    double* mb = (double*)malloc(sizeof(double) * (size_t)n);
    double cur = floor((t[0] - t[0]) / D), acc = 0.0, inv = 0.0;
    int64_t cnt = 0;
    for (int64_t i = 0; i < n; ++i) {
      double b = floor((t[i] - t[0]) / D);
      if (b != cur) { mb[nbins++] = acc / (double)cnt; inv += 1.0 / (double)cnt; cur = b; acc = 0.0; cnt = 0; }
      acc += r[i]; ++cnt;
    }
    mb[nbins++] = acc / (double)cnt; inv += 1.0 / (double)cnt;
    double msum = 0.0;
    for (int32_t b = 0; b < nbins; ++b) msum += mb[b];
    double mbar = msum / (double)nbins, s2 = 0.0;
    for (int32_t b = 0; b < nbins; ++b) s2 += (mb[b] - mbar) * (mb[b] - mbar);
    var_bin = s2 / (double)nbins;
    mean_inv = inv / (double)nbins;
    free(mb);
  }
  double var_r = var_bin - var_w * mean_inv;
  if (var_r < 0.0) var_r = 0.0;
  out->sigma_w = sqrt(var_w); out->sigma_r = sqrt(var_r);
  out->depth_eff = delta * (1.0 - qin);
  out->n_t = n_t; out->n_transits = n_tr; out->n_bins = nbins;
  double den = 0.0;
  if (n_t > 0 && n_tr > 0) den = var_w / (double)n_t + var_r / (double)n_tr;
  out->snr_pink = den > 0.0 ? out->depth_eff / sqrt(den) : 0.0;
  out->detected = (n_tr >= 2 && out->snr_pink > 9.0 && snr > 9.0) ? 1 : 0;
  free(r);
}
int orc_sizeof_pink(void) { return (int)sizeof(orc_pink); }
