/*
 * gbk_oracle.c -- CPU ORACLE.  TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * A plain, slow, double-precision restatement of the intensity-cube modelling
 * strategy of Bekiaris et al. (arXiv:1510.01815, "GBKFIT"), written from
 * /root/reference/PAPER.md.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may build, load or call it.
 * It shares no code, header, table or constant generator with the CUDA path
 * under paper_1510_01815_b200/csrc/, and neither side includes the other.
 *
 * The method is a definition, not an approximation, so the oracle is that
 * definition written out literally, in the paper's order (PAPER.md:63-66 and
 * sections 2.2.2-2.2.6):
 *
 *   1. evaluate the model cube (eq. 1-8 + Gaussian line)       gbko_model_cube
 *   2. convolve with the LSF along v (direct sum)               gbko_conv_lsf
 *   3. convolve with the PSF in (x,y), per channel (direct sum) gbko_conv_psf
 *   4. down-sample by the up-sampling factor u                  gbko_downsample
 *   5. zeroth/first/second moments of every spectrum            gbko_moments
 *   6. masked, error-weighted chi^2 (eq. 11)                    gbko_chi2
 *
 * There is no blocking, fusion, separable-pass trick, FFT or moment-first
 * shortcut: the convolution of the paper's FFT step reaches
 * exactly the linear convolution, whose plain definition is the direct sum
 * used here.  OpenMP is used over independent parameter rows only.
 *
 * Readings of the paper where it is silent (A1..A16):
 *   A1  pixel j has centre coordinate j; fine sample a of an up-sampled grid
 *       sits at x_a = (a + 0.5)/u - 0.5.
 *   A2  channel k has velocity v_k = v_center + (k - (nv-1)/2) * dv.
 *   A3  line(c) = I * dv/(sigma0*sqrt(2 pi)) * exp(-(v_c - v_los)^2/(2 sigma0^2))
 *       (flux-normalised point sample).
 *   A4  m0 = plain sum over in-band channels.
 *   A6  the model is evaluated in the halo needed by the two "valid"
 *       convolutions (R_p fine pixels in x,y; R_v channels in v);
 *       halo_zero=1 replaces those values by zero (unit tests only).
 *   A7  linear ramp: V_rot = V_t * min(r/r_t, 1).
 *   A8  r = 0  =>  cos(theta) := 0.
 *   A9  taps are renormalised to sum exactly 1 (by the caller / tap builders).
 *   A11 true convolution (kernel flipped).
 *   A15 a row is out of domain (chi^2 = +INF, maps NaN) when a parameter is
 *       non-finite, sigma0 <= 0, r0 <= 0, r_t <= 0, I0 <= 0 or |cos i| < 1e-6;
 *       an unmasked spaxel with m0 < 1e-30 * I0 ("model-dark") or non-finite
 *       moments makes the row's chi^2 +INF.
 *
 * PARITY PINS: every exported step is pinned by tests/test_oracle_pins.py
 * against closed forms, hand values, invariants and brute force (see
 * DESIGN.md "What pins the oracle").  The conventions A1-A4, A6, A9, A10 are
 * choices the paper does not fix: for those, "parity unpinned" by the paper.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define GBKO_P 10 /* xo, yo, pa_deg, inc_deg, vsys, vt, rt, sigma0, r0, i0 */
#define GBKO_P_EPINAT 12 /* ... + a, g: the slopes of eq. 7 */
#define GBKO_PI 3.14159265358979323846

typedef struct {
  int32_t nx, ny, nv;  /* observed grid: spaxels and channels              */
  int32_t u;           /* spatial up-sampling factor        */
  double v_center, dv; /* A2                                               */
  int32_t rc_model;    /* 0 = arctan (eq. 6), 1 = linear ramp (A7), 2 = Epinat (eq. 7): rows of 12 */
  int32_t psf_n;       /* odd side of the PSF image on the fine grid       */
  const double *psf;   /* [psf_n*psf_n], row-major (y, x), sum = 1         */
  int32_t lsf_n;       /* odd length of the LSF taps (channels)            */
  const double *lsf;   /* [lsf_n], sum = 1                                 */
  int32_t halo_zero;   /* A6 switch, unit tests only                       */
  /* "User-specified intensity model" (reading A22 of DESIGN.md): when tab_n > 0 the
   * radial profile of eq. 5 is replaced by I(r) = I0 * T(r / r0), T tabulated at x_j = j * tab_dx,
   * j = 0..tab_n-1, linear interpolation between nodes, T = tab[tab_n-1] beyond the last node.   */
  int32_t tab_n;
  const double *tab;
  double tab_dx;
  int32_t extract;     /* 0: moments (the paper's choice); 1: Gaussian-profile fit of every spectrum  */
                       /* ("fitting an analytic profile (e.g., Gaussian)"; reading A23)  */
} gbko_grid;

/* Parameters per row: 12 with the Epinat curve, else 10.                      */
int gbko_row_len(int rc_model) { return rc_model == 2 ? GBKO_P_EPINAT : GBKO_P; }

/* ---------------------------------------------------------------- taps -- */

/* Gaussian taps g[j] = exp(-j^2/(2 sigma^2)), j in [-R, R], R = ceil(4 sigma),
 * normalised to sum 1 (eq. 9 sampled; A9, A10).  sigma <= 0
 * gives the delta kernel (R = 0).  Returns R, or -1 if cap is too small.  */
int gbko_gaussian_taps(double sigma, double *taps, int cap) {
  if (!(sigma > 0.0)) {
    if (cap < 1) return -1;
    taps[0] = 1.0;
    return 0;
  }
  int R = (int)ceil(4.0 * sigma);
  if (2 * R + 1 > cap) return -1;
  double s = 0.0;
  for (int j = -R; j <= R; ++j) {
    taps[j + R] = exp(-0.5 * (double)j * (double)j / (sigma * sigma));
    s += taps[j + R];
  }
  for (int j = 0; j <= 2 * R; ++j) taps[j] /= s;
  return R;
}

/* FWHM -> sigma of a Gaussian: sigma = FWHM / (2 sqrt(2 ln 2)).            */
double gbko_fwhm_to_sigma(double fwhm) { return fwhm / (2.0 * sqrt(2.0 * log(2.0))); }

/* 2-D Gaussian PSF image on the fine grid = outer product of the 1-D taps
 * with sigma_f = u * sigma (eq. 9 spatial part; A14).  Returns n = 2R+1.    */
int gbko_psf_gaussian_image(double fwhm_data_px, int u, double *img, int cap_side) {
  double t[1024];
  int R = gbko_gaussian_taps((double)u * gbko_fwhm_to_sigma(fwhm_data_px), t, 1024);
  if (R < 0 || 2 * R + 1 > cap_side) return -1;
  int n = 2 * R + 1;
  for (int y = 0; y < n; ++y)
    for (int x = 0; x < n; ++x) img[y * n + x] = t[y] * t[x];
  return n;
}

/* Moffat PSF image P ~ [1 + (jx^2+jy^2)/alpha^2]^(-beta),
 * alpha = FWHM / (2 sqrt(2^(1/beta) - 1)), point-sampled at integer fine-pixel
 * offsets on an n x n grid (n odd), normalised to sum 1 (A9).               */
int gbko_psf_moffat_image(double fwhm_fine_px, double beta, int n, double *img) {
  if (n < 1 || (n & 1) == 0) return -1;
  int R = n / 2;
  double alpha = fwhm_fine_px / (2.0 * sqrt(pow(2.0, 1.0 / beta) - 1.0));
  double s = 0.0;
  for (int y = -R; y <= R; ++y)
    for (int x = -R; x <= R; ++x) {
      double v = pow(1.0 + ((double)x * x + (double)y * y) / (alpha * alpha), -beta);
      img[(y + R) * n + (x + R)] = v;
      s += v;
    }
  for (int k = 0; k < n * n; ++k) img[k] /= s;
  return n;
}

/* ------------------------------------------------------- disc model ---- */

/* Domain rule A15.  Returns 1 when the row can be evaluated.                */
int gbko_row_valid(const double *p) {
  for (int k = 0; k < GBKO_P; ++k)
    if (!isfinite(p[k])) return 0;
  if (!(p[7] > 0.0) || !(p[8] > 0.0) || !(p[6] > 0.0) || !(p[9] > 0.0)) return 0;
  if (fabs(cos(p[3] * GBKO_PI / 180.0)) < 1e-6) return 0;
  return 1;
}

/* The same for a row of the given rotation curve: the Epinat slopes a = p[10],
 * g = p[11] must be finite and > 0 as well.                                   */
int gbko_row_valid_rc(const double *p, int rc_model) {
  if (!gbko_row_valid(p)) return 0;
  if (rc_model == 2 && (!isfinite(p[10]) || !isfinite(p[11]) || !(p[10] > 0.0) || !(p[11] > 0.0)))
    return 0;
  return 1;
}

/* Tabulated radial profile T(x), x = r / r0 (see gbko_grid).                 */
double gbko_table_profile(const double *tab, int n, double dx, double x) {
  const double t = x / dx;
  if (!(t < (double)(n - 1))) return tab[n - 1];
  const int j = (int)floor(t);
  const double f = t - (double)j;
  return tab[j] + f * (tab[j + 1] - tab[j]);
}

/* One sky position (x, y): eq. 1-4 (deprojection), eq. 5 (brightness),
 * eq. 6 or the ramp (rotation curve), eq. 8 (line-of-sight velocity).
 * PAPER.md:84-96, 110, 120, 143.                                           */
void gbko_disc_point(const double *p, int rc_model, double x, double y, double *I_out,
                     double *vlos_out) {
  const double xo = p[0], yo = p[1];
  const double pa = p[2] * GBKO_PI / 180.0, inc = p[3] * GBKO_PI / 180.0;
  const double vsys = p[4], vt = p[5], rt = p[6], r0 = p[8], i0 = p[9];
  const double sp = sin(pa), cp = cos(pa), si = sin(inc), ci = cos(inc);
  const double xe = -(x - xo) * sp + (y - yo) * cp;     /* eq. 1 */
  const double ye = -(x - xo) * cp - (y - yo) * sp;     /* eq. 2 */
  const double yd = ye / ci;
  const double r = sqrt(xe * xe + yd * yd);             /* eq. 3 */
  const double cos_theta = (r > 0.0) ? xe / r : 0.0;    /* eq. 4, A8 */
  const double I = i0 * exp(-r / r0);                   /* eq. 5 */
  double vrot;
  if (rc_model == 0)
    vrot = (2.0 / GBKO_PI) * vt * atan(r / rt);         /* eq. 6 */
  else if (rc_model == 1)
    vrot = vt * fmin(r / rt, 1.0);                      /* A7 */
  else                                                  /* eq. 7: a = p[10], g = p[11] */
    vrot = vt * pow(r / rt, p[11]) / (1.0 + pow(r / rt, p[10]));
  *I_out = I;
  *vlos_out = vsys + vrot * si * cos_theta;             /* eq. 8 */
}

/* Channel velocity, A2; c may lie outside [0, nv) (spectral halo).          */
double gbko_channel_velocity(const gbko_grid *g, int c) {
  return g->v_center + ((double)c - 0.5 * (double)(g->nv - 1)) * g->dv;
}

/* Fine-grid coordinate of fine index a (may be negative: spatial halo), A1. */
double gbko_fine_coord(int a, int u) { return ((double)a + 0.5) / (double)u - 0.5; }

/* Sizes of the extended (halo-carrying) cube.                               */
void gbko_ext_dims(const gbko_grid *g, int *ew, int *eh, int *ec) {
  *ew = g->u * g->nx + (g->psf_n - 1);
  *eh = g->u * g->ny + (g->psf_n - 1);
  *ec = g->nv + (g->lsf_n - 1);
}

/* Step 1 (section 2.2.2): the model cube on the extended grid,
 * layout cube[c][b][a] (a = x fastest, then y, then v -- slice-major as in
 * PAPER.md:234).  Index (c, b, a) holds channel c - R_v, fine pixel
 * (a - R_p, b - R_p).                                                      */
void gbko_model_cube(const gbko_grid *g, const double *p, double *cube) {
  int ew, eh, ec;
  gbko_ext_dims(g, &ew, &eh, &ec);
  const int Rp = g->psf_n / 2, Rv = g->lsf_n / 2;
  const double sigma0 = p[7];
  const double amp = g->dv / (sigma0 * sqrt(2.0 * GBKO_PI)); /* A3 */
  for (int b = 0; b < eh; ++b)
    for (int a = 0; a < ew; ++a) {
      const int fa = a - Rp, fb = b - Rp;
      const int in_field = fa >= 0 && fa < g->u * g->nx && fb >= 0 && fb < g->u * g->ny;
      double I, vlos;
      const double xs = gbko_fine_coord(fa, g->u), ys = gbko_fine_coord(fb, g->u);
      gbko_disc_point(p, g->rc_model, xs, ys, &I, &vlos);
      if (g->tab_n > 0) {          /* user-specified profile instead of eq. 5: I0 * T(r / r0) */
        const double pa = p[2] * GBKO_PI / 180.0, inc = p[3] * GBKO_PI / 180.0;
        const double xe = -(xs - p[0]) * sin(pa) + (ys - p[1]) * cos(pa);   /* eq. 1 */
        const double ye = -(xs - p[0]) * cos(pa) - (ys - p[1]) * sin(pa);   /* eq. 2 */
        const double r = sqrt(xe * xe + (ye / cos(inc)) * (ye / cos(inc))); /* eq. 3 */
        I = p[9] * gbko_table_profile(g->tab, g->tab_n, g->tab_dx, r / p[8]);
      }
      for (int c = 0; c < ec; ++c) {
        const int ch = c - Rv;
        const int in_band = ch >= 0 && ch < g->nv;
        double val;
        if (g->halo_zero && !(in_field && in_band)) {
          val = 0.0;
        } else {
          const double dvel = gbko_channel_velocity(g, ch) - vlos;
          val = I * amp * exp(-0.5 * dvel * dvel / (sigma0 * sigma0));
        }
        cube[((size_t)c * eh + b) * ew + a] = val;
      }
    }
}

/* Step 2: LSF, direct "valid" convolution along v (true convolution, A11):
 * out[k] = sum_{t=0}^{n-1} L[t] * in[k + (n-1) - t],  k in [0, nc_in-n+1).
 * in: [nc_in][plane], out: [nc_in - n + 1][plane].                         */
void gbko_conv_lsf(const double *in, int nc_in, size_t plane, const double *L, int n,
                   double *out) {
  const int nc_out = nc_in - n + 1;
  for (int k = 0; k < nc_out; ++k)
    for (size_t q = 0; q < plane; ++q) {
      double s = 0.0;
      for (int t = 0; t < n; ++t) s += L[t] * in[(size_t)(k + (n - 1) - t) * plane + q];
      out[(size_t)k * plane + q] = s;
    }
}

/* Step 3: PSF, direct "valid" 2-D convolution per channel (true convolution):
 * out[b][a] = sum_{ty,tx} P[ty][tx] * in[b + (n-1) - ty][a + (n-1) - tx].
 * in: [nch][eh][ew], out: [nch][eh-n+1][ew-n+1].      */
void gbko_conv_psf(const double *in, int nch, int eh, int ew, const double *P, int n,
                   double *out) {
  const int oh = eh - n + 1, ow = ew - n + 1;
  for (int c = 0; c < nch; ++c) {
    const double *src = in + (size_t)c * eh * ew;
    double *dst = out + (size_t)c * oh * ow;
    for (int b = 0; b < oh; ++b)
      for (int a = 0; a < ow; ++a) {
        double s = 0.0;
        for (int ty = 0; ty < n; ++ty)
          for (int tx = 0; tx < n; ++tx)
            s += P[ty * n + tx] * src[(size_t)(b + (n - 1) - ty) * ew + (a + (n - 1) - tx)];
        dst[(size_t)b * ow + a] = s;
      }
  }
}

/* Step 4: mean over each u x u block of fine pixels.
 * in: [nch][fh][fw] with fh = u*ny, fw = u*nx; out: [nch][ny][nx].          */
void gbko_downsample(const double *in, int nch, int ny, int nx, int u, double *out) {
  const int fh = u * ny, fw = u * nx;
  for (int c = 0; c < nch; ++c)
    for (int y = 0; y < ny; ++y)
      for (int x = 0; x < nx; ++x) {
        double s = 0.0;
        for (int dy = 0; dy < u; ++dy)
          for (int dx = 0; dx < u; ++dx)
            s += in[((size_t)c * fh + (size_t)(u * y + dy)) * fw + (size_t)(u * x + dx)];
        out[((size_t)c * ny + y) * nx + x] = s / (double)(u * u);
      }
}

/* Step 5 (A4, A5): per spectrum
 *   m0 = sum_k C_k,  m1 = sum_k C_k v_k / m0,
 *   m2 = sqrt(max(0, sum_k C_k (v_k - m1)^2 / m0)).
 * cube: [nv][npix]; vel: [nv].  m0 == 0 gives NaN moments (0/0).           */
void gbko_moments(const double *cube, int nv, size_t npix, const double *vel, double *m0,
                  double *m1, double *m2) {
  for (size_t q = 0; q < npix; ++q) {
    double s0 = 0.0, s1 = 0.0;
    for (int k = 0; k < nv; ++k) {
      const double c = cube[(size_t)k * npix + q];
      s0 += c;
      s1 += c * vel[k];
    }
    const double mean = s1 / s0;
    double s2 = 0.0;
    for (int k = 0; k < nv; ++k) {
      const double d = vel[k] - mean;
      s2 += cube[(size_t)k * npix + q] * d * d;
    }
    m0[q] = s0;
    m1[q] = mean;
    const double var = s2 / s0;
    m2[q] = isnan(var) ? NAN : sqrt(fmax(0.0, var)); /* fmax would hide a NaN */
  }
}

/* Step 5, the alternative the paper describes and times but does not adopt (PAPER.md:228-232,
 * 493-507, 666-678): fit G(v) = A exp(-(v - mu)^2 / (2 s^2)) to every spectrum by unweighted least
 * squares; velocity = mu, dispersion = s; m0 stays the plain sum (A4).  Reading A23 of DESIGN.md (the
 * paper used MPFIT and gives no details): Levenberg-Marquardt on (A, mu, s),
 *   start   mu = m1, s = max(m2, dv/2), A = m0 dv / (s sqrt(2 pi))   (from the moments)
 *   step    (J^T J + lambda diag(J^T J)) delta = J^T r,  r_k = C_k - G(v_k), lambda_0 = 1e-3
 *   accept  when the sum of squares decreases: lambda <- max(lambda/10, 1e-12); else lambda <- 10 lambda
 *   stop    converged when an accepted step has |delta mu| and |delta s| < 1e-6 dv, or when the sum of
 *           squares is already <= 1e-28 m0^2 (an exact fit); FAILED (NaN velocity and dispersion: "may
 *           occasionally fail to converge") after 200 iterations, when lambda exceeds
 *           1e12, when s leaves (0, 1e3 nv dv) or a value is not finite.
 * A spectrum with m0 == 0 or non-finite moments gives NaN.                                        */
void gbko_gaussfit(const double *cube, int nv, size_t npix, const double *vel, double *m0,
                   double *mu_out, double *s_out) {
  const double dv = nv > 1 ? vel[1] - vel[0] : 1.0;
  for (size_t q = 0; q < npix; ++q) {
    double s0 = 0.0, s1 = 0.0;
    for (int k = 0; k < nv; ++k) {
      const double c = cube[(size_t)k * npix + q];
      s0 += c;
      s1 += c * vel[k];
    }
    const double mean = s1 / s0;
    double s2 = 0.0;
    for (int k = 0; k < nv; ++k) {
      const double d = vel[k] - mean;
      s2 += cube[(size_t)k * npix + q] * d * d;
    }
    m0[q] = s0;
    mu_out[q] = s_out[q] = NAN;
    const double var = s2 / s0;
    if (!(s0 > 0.0) || !isfinite(mean) || !isfinite(var)) continue;
    double mu = mean, sg = fmax(sqrt(fmax(var, 0.0)), 0.5 * dv);
    double A = s0 * dv / (sg * sqrt(2.0 * GBKO_PI));
    double lambda = 1e-3;
    int done = 0;
    for (int it = 0; it < 200 && !done; ++it) {
      /* normal equations at (A, mu, sg) */
      double JJ[3][3] = {{0, 0, 0}, {0, 0, 0}, {0, 0, 0}}, Jr[3] = {0, 0, 0}, sse = 0.0;
      for (int k = 0; k < nv; ++k) {
        const double d = vel[k] - mu;
        const double e = exp(-0.5 * d * d / (sg * sg));
        const double r = cube[(size_t)k * npix + q] - A * e;
        const double J[3] = {e, A * e * d / (sg * sg), A * e * d * d / (sg * sg * sg)};
        for (int a = 0; a < 3; ++a) {
          Jr[a] += J[a] * r;
          for (int b = 0; b < 3; ++b) JJ[a][b] += J[a] * J[b];
        }
        sse += r * r;
      }
      if (sse <= 1e-28 * s0 * s0) {
        done = 1;
        break;
      }
      /* damped solve by Cramer's rule (3 x 3) */
      double M[3][3];
      for (int a = 0; a < 3; ++a)
        for (int b = 0; b < 3; ++b) M[a][b] = JJ[a][b] * (a == b ? 1.0 + lambda : 1.0);
      const double det = M[0][0] * (M[1][1] * M[2][2] - M[1][2] * M[2][1]) -
                         M[0][1] * (M[1][0] * M[2][2] - M[1][2] * M[2][0]) +
                         M[0][2] * (M[1][0] * M[2][1] - M[1][1] * M[2][0]);
      double dl[3];
      for (int c = 0; c < 3; ++c) {
        double N[3][3];
        for (int a = 0; a < 3; ++a)
          for (int b = 0; b < 3; ++b) N[a][b] = b == c ? Jr[a] : M[a][b];
        dl[c] = (N[0][0] * (N[1][1] * N[2][2] - N[1][2] * N[2][1]) -
                 N[0][1] * (N[1][0] * N[2][2] - N[1][2] * N[2][0]) +
                 N[0][2] * (N[1][0] * N[2][1] - N[1][1] * N[2][0])) / det;
      }
      const double A1 = A + dl[0], mu1 = mu + dl[1], sg1 = sg + dl[2];
      double sse1 = INFINITY;
      if (isfinite(A1) && isfinite(mu1) && sg1 > 0.0 && sg1 < 1e3 * nv * dv) {
        sse1 = 0.0;
        for (int k = 0; k < nv; ++k) {
          const double d = vel[k] - mu1;
          const double r = cube[(size_t)k * npix + q] - A1 * exp(-0.5 * d * d / (sg1 * sg1));
          sse1 += r * r;
        }
      }
      if (sse1 < sse) {
        A = A1, mu = mu1, sg = sg1;
        lambda = fmax(lambda / 10.0, 1e-12);
        if (fabs(dl[1]) < 1e-6 * dv && fabs(dl[2]) < 1e-6 * dv) done = 1;
      } else {
        lambda *= 10.0;
        if (!(lambda <= 1e12)) break;
      }
    }
    if (done) mu_out[q] = mu, s_out[q] = sg;
  }
}

/* Step 6 (eq. 11; masks PAPER.md:185): W is pre-folded
 * into serr by the caller; sobs == NULL drops the dispersion term.
 * Optional resid[2][npix] receives the weighted residuals (0 where masked,
 * and 0 for the dispersion plane when sobs == NULL).
 * dark_level: an unmasked spaxel with m0 < dark_level, or with non-finite
 * m1/m2, makes the result +INF (A15).                                       */
double gbko_chi2(const double *m0, const double *m1, const double *m2, const float *vobs,
                 const float *verr, const float *sobs, const float *serr, const uint8_t *mask,
                 size_t npix, double dark_level, double *resid) {
  double chi2 = 0.0;
  int bad = 0;
  for (size_t q = 0; q < npix; ++q) {
    double t = 0.0, s = 0.0;
    if (!mask || mask[q]) {
      if (!(m0[q] >= dark_level) || !isfinite(m1[q]) || !isfinite(m2[q])) {
        bad = 1;
        t = s = NAN;
      } else {
        t = (m1[q] - (double)vobs[q]) / (double)verr[q];
        if (sobs) s = (m2[q] - (double)sobs[q]) / (double)serr[q];
        chi2 += t * t + s * s;
      }
    }
    if (resid) {
      resid[q] = t;
      resid[npix + q] = s;
    }
  }
  return bad ? INFINITY : chi2;
}

/* ------------------------------------------------------ whole pipeline -- */

/* Moment maps of one parameter row: steps 1-5.  Work buffers are allocated
 * here (the oracle is not tuned).  Returns 0, or -1 on allocation failure.
 * An out-of-domain row fills the maps with NaN and returns 1.              */
int gbko_model_maps(const gbko_grid *g, const double *p, double *m0, double *m1, double *m2) {
  const size_t npix = (size_t)g->nx * g->ny;
  if (!gbko_row_valid_rc(p, g->rc_model)) {
    for (size_t q = 0; q < npix; ++q) m0[q] = m1[q] = m2[q] = NAN;
    return 1;
  }
  int ew, eh, ec;
  gbko_ext_dims(g, &ew, &eh, &ec);
  const int fw = g->u * g->nx, fh = g->u * g->ny;
  double *cube = (double *)malloc(sizeof(double) * (size_t)ec * eh * ew);
  double *c_lsf = (double *)malloc(sizeof(double) * (size_t)g->nv * eh * ew);
  double *c_psf = (double *)malloc(sizeof(double) * (size_t)g->nv * fh * fw);
  double *c_ds = (double *)malloc(sizeof(double) * (size_t)g->nv * npix);
  double *vel = (double *)malloc(sizeof(double) * (size_t)g->nv);
  int rc = -1;
  if (cube && c_lsf && c_psf && c_ds && vel) {
    gbko_model_cube(g, p, cube);                                     /* 1 */
    gbko_conv_lsf(cube, ec, (size_t)eh * ew, g->lsf, g->lsf_n, c_lsf); /* 2 */
    gbko_conv_psf(c_lsf, g->nv, eh, ew, g->psf, g->psf_n, c_psf);    /* 3 */
    gbko_downsample(c_psf, g->nv, g->ny, g->nx, g->u, c_ds);         /* 4 */
    for (int k = 0; k < g->nv; ++k) vel[k] = gbko_channel_velocity(g, k);
    if (g->extract == 1)
      gbko_gaussfit(c_ds, g->nv, npix, vel, m0, m1, m2);             /* 5, Gaussian-fit variant */
    else
      gbko_moments(c_ds, g->nv, npix, vel, m0, m1, m2);              /* 5 */
    rc = 0;
  }
  free(cube);
  free(c_lsf);
  free(c_psf);
  free(c_ds);
  free(vel);
  return rc;
}

/* K parameter rows (float32 at the boundary, promoted to double; gbko_row_len
 * floats each) against one observed data set.  Outputs (any may be NULL except chi2):
 *   chi2[K]; m0,m1,m2[K][ny][nx]; resid[K][2][ny][nx].
 * nthreads <= 0 uses the OpenMP default.  Returns 0 or -1.                  */
int gbko_eval_rows(const gbko_grid *g, const float *vobs, const float *verr, const float *sobs,
                   const float *serr, const uint8_t *mask, const float *params, int64_t K,
                   double *chi2, double *m0, double *m1, double *m2, double *resid,
                   int nthreads) {
  const size_t npix = (size_t)g->nx * g->ny;
  int fail = 0;
#ifdef _OPENMP
  if (nthreads > 0) omp_set_num_threads(nthreads);
#else
  (void)nthreads;
#endif
  const int P = gbko_row_len(g->rc_model);
#pragma omp parallel for schedule(dynamic, 1)
  for (int64_t k = 0; k < K; ++k) {
    double p[GBKO_P_EPINAT];
    for (int j = 0; j < P; ++j) p[j] = (double)params[k * P + j];
    double *a0 = (double *)malloc(sizeof(double) * npix * 3);
    if (!a0) {
      fail = 1;
      continue;
    }
    double *a1 = a0 + npix, *a2 = a1 + npix;
    const int st = gbko_model_maps(g, p, a0, a1, a2);
    if (st < 0) fail = 1;
    double *r = resid ? resid + (size_t)k * 2 * npix : NULL;
    if (st == 1) {
      chi2[k] = INFINITY;
      if (r)
        for (size_t q = 0; q < 2 * npix; ++q) r[q] = NAN;
    } else {
      chi2[k] = gbko_chi2(a0, a1, a2, vobs, verr, sobs, serr, mask, npix, 1e-30 * p[9], r);
    }
    if (m0) memcpy(m0 + (size_t)k * npix, a0, sizeof(double) * npix);
    if (m1) memcpy(m1 + (size_t)k * npix, a1, sizeof(double) * npix);
    if (m2) memcpy(m2 + (size_t)k * npix, a2, sizeof(double) * npix);
    free(a0);
  }
  return fail ? -1 : 0;
}

/* ---------------------------------------------------- velocity field ---- */

/* Velocity-field modelling strategy (section 2.2.1): eq. 8
 * evaluated at every spaxel centre (x = column, y = row; reading A1), no cube,
 * no PSF, no LSF (the paper skips steps 2.2.2-2.2.5), then the
 * velocity residual and the first term of eq. 11 only
 * (no dispersion map is modelled).  Only the seven kinematic
 * parameters p[0..6] are used (plus a = p[10], g = p[11] of the 12-float rows
 * of the Epinat curve, rc_model 2, eq. 7); a row is out of domain when one of
 * them is not finite,
 * r_t <= 0, |cos i| < 1e-6, or a <= 0 or g <= 0 (chi2 = +INF, NaN maps).
 * Outputs: chi2[K]; vmap[K][ny][nx] and resid[K][ny][nx] may be NULL.        */
int gbko_vfield_rows(const gbko_grid *g, const float *vobs, const float *verr, const uint8_t *mask,
                     const float *params, int64_t K, double *chi2, double *vmap, double *resid,
                     int nthreads) {
  const size_t npix = (size_t)g->nx * g->ny;
#ifdef _OPENMP
  if (nthreads > 0) omp_set_num_threads(nthreads);
#else
  (void)nthreads;
#endif
  const int P = gbko_row_len(g->rc_model);
#pragma omp parallel for schedule(dynamic, 16)
  for (int64_t k = 0; k < K; ++k) {
    double p[GBKO_P_EPINAT];
    int ok = 1;
    for (int j = 0; j < P; ++j) p[j] = (double)params[k * P + j];
    for (int j = 0; j < 7; ++j)
      if (!isfinite(p[j])) ok = 0;
    if (ok && (!(p[6] > 0.0) || fabs(cos(p[3] * GBKO_PI / 180.0)) < 1e-6)) ok = 0;
    if (g->rc_model == 2) {               /* Epinat curve: the slopes a = p[10], g = p[11] must be > 0 */
      if (!isfinite(p[10]) || !isfinite(p[11]) || !(p[10] > 0.0) || !(p[11] > 0.0)) ok = 0;
      if (!ok) p[10] = 1.0, p[11] = 1.0;
    }
    p[7] = 1.0, p[8] = 1.0, p[9] = 1.0;   /* sigma0, r0, I0 are not part of eq. 8; keep the brightness finite */
    double sum = 0.0;
    for (size_t q = 0; q < npix; ++q) {
      const int iy = (int)(q / (size_t)g->nx), ix = (int)(q % (size_t)g->nx);
      double I, v = NAN;
      if (ok) gbko_disc_point(p, g->rc_model, (double)ix, (double)iy, &I, &v);
      const int unmasked = !mask || mask[q] != 0;
      double t = 0.0;
      if (unmasked) {
        t = (v - (double)vobs[q]) / (double)verr[q];
        if (!isfinite(t)) sum = INFINITY; else if (isfinite(sum)) sum += t * t;
      }
      if (vmap) vmap[(size_t)k * npix + q] = v;
      if (resid) resid[(size_t)k * npix + q] = unmasked ? (ok ? t : NAN) : 0.0;
    }
    chi2[k] = ok ? sum : INFINITY;
  }
  return 0;
}

int gbko_max_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}
