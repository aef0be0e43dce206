/*
 * gbk_cpu_fast.c -- an OPTIMISED CPU restatement, for TIMING ONLY.  TEST / BENCH INFRASTRUCTURE,
 * NOT PRODUCT CODE and NOT THE ORACLE.
 *
 * bench.py's cpu_baseline times the parity oracle (gbk_oracle.c) as it stands: the paper's
 * definition written out literally in FP64, with a materialised cube and a direct 2-D PSF sum per
 * channel.  A GPU / oracle ratio therefore compares a tuned kernel with a deliberately naive
 * program.  This file is the straightforward fast CPU version a practitioner would write, so that
 * a second, clearly labelled baseline ("kind": "optimised-cpu") stands beside it:
 *   - float32 throughout;
 *   - the moment-first identity: S_q = PSF (*) sum_c w_q[c] line(x, y, c), q = 0, 1, 2, with the LSF
 *     folded into the channel weights w_q (the cube is never stored; only three maps are convolved);
 *   - separable Gaussian PSF passes;
 *   - OpenMP over rows, inner channel loop written for auto-vectorisation (gcc -O3 -ffast-math
 *     -march=native, expf through libmvec).
 * It covers what the headline configs need (arctan or ramp curve, exponential disc, Gaussian PSF,
 * Gaussian LSF, any up-sampling) and nothing else.  tests/test_cpu_fast.py checks it against the
 * oracle at BASELINE.json's tolerances.  It shares no code with the CUDA path or with the oracle;
 * only tests/ and bench.py's cpu_baseline leg may build or call it.
 *
 * Equations: PAPER.md:84-96 (eq. 1-4), :110 (eq. 5), :120 (eq. 6), :143 (eq. 8), :199 (line),
 * :214-218 (PSF, LSF), :222 (down-sampling), :228-234 (moments), :246 (eq. 11); readings A1-A16 of
 * DESIGN.md as in the oracle.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef struct {
  int32_t nx, ny, nv, u;
  float v_center, dv;
  int32_t rc_model;     /* 0 arctan, 1 ramp */
  int32_t r_p;          /* PSF tap radius on the fine grid */
  const float *psf;     /* [2 r_p + 1] 1-D Gaussian taps, sum 1 */
  int32_t r_v;          /* LSF tap radius */
  const float *lsf;     /* [2 r_v + 1], sum 1 */
} gbkf_grid;

static int row_ok(const float *p) {
  for (int j = 0; j < 10; ++j)
    if (!isfinite(p[j])) return 0;
  if (!(p[7] > 0.f) || !(p[8] > 0.f) || !(p[6] > 0.f) || !(p[9] > 0.f)) return 0;
  if (fabs(cos((double)p[3] * 3.14159265358979323846 / 180.0)) < 1e-6) return 0;
  return 1;
}

/* K float32 rows of 10 parameters against one observed data set -> chi2[K].  Returns 0, or -1 on
 * allocation failure.                                                                            */
int gbkf_eval_rows(const gbkf_grid *g, const float *vobs, const float *verr, const float *sobs,
                   const float *serr, const uint8_t *mask, const float *params, int64_t K,
                   float *chi2, int nthreads) {
  const int u = g->u, R = g->r_p, Rv = g->r_v;
  const int fw = u * g->nx, fh = u * g->ny, EW = fw + 2 * R, EH = fh + 2 * R, nvx = g->nv + 2 * Rv;
  const float vhalf = 0.5f * (float)(g->nv - 1) * g->dv;
  int fail = 0;
#ifdef _OPENMP
  if (nthreads > 0) omp_set_num_threads(nthreads);
#else
  (void)nthreads;
#endif
#pragma omp parallel
  {
    float *S = (float *)malloc(sizeof(float) * 3 * (size_t)EW * EH);   /* S0, S1, S2 on the extended grid */
    float *T = (float *)malloc(sizeof(float) * 3 * (size_t)fw * EH);   /* after the x pass */
    float *w = (float *)malloc(sizeof(float) * 4 * (size_t)nvx);       /* v_c, w0, w1, w2 */
    if (!S || !T || !w) fail = 1;
#pragma omp for schedule(dynamic, 1)
    for (int64_t k = 0; k < K; ++k) {
      if (fail) continue;
      const float *p = params + k * 10;
      if (!row_ok(p)) {
        chi2[k] = INFINITY;
        continue;
      }
      const float xo = p[0], yo = p[1], vsys = p[4] - g->v_center, vt = p[5], rt = p[6];
      const float sig = p[7], r0 = p[8], i0 = p[9];
      const double pa = (double)p[2] * 3.14159265358979323846 / 180.0, inc = (double)p[3] * 3.14159265358979323846 / 180.0;
      const float sp = (float)sin(pa), cp = (float)cos(pa), si = (float)sin(inc), inv_ci = (float)(1.0 / cos(inc));
      const float v_ref = fminf(fmaxf(vsys, -vhalf), vhalf);   /* moments about a velocity near the line */
      /* channel table: velocity (from v_ref) and LSF-folded weights of every extended channel */
      float *vc = w, *w0 = w + nvx, *w1 = w + 2 * nvx, *w2 = w + 3 * nvx;
      for (int c = 0; c < nvx; ++c) {
        const int ch = c - Rv;
        double a0 = 0, a1 = 0, a2 = 0;
        for (int kk = ch - Rv < 0 ? 0 : ch - Rv; kk <= (ch + Rv > g->nv - 1 ? g->nv - 1 : ch + Rv); ++kk) {
          const double L = g->lsf[(kk - ch) + Rv];
          const double v = ((double)kk - 0.5 * (g->nv - 1)) * (double)g->dv - (double)v_ref;
          a0 += L, a1 += L * v, a2 += L * v * v;
        }
        vc[c] = ((float)ch - 0.5f * (float)(g->nv - 1)) * g->dv;   /* from v_center */
        w0[c] = (float)a0, w1[c] = (float)a1, w2[c] = (float)a2;
      }
      const float amp = g->dv / (sig * 2.5066282746310002f) / (float)(u * u);
      const float inv2s2 = -0.5f / (sig * sig);
      for (int b = 0; b < EH; ++b) {
        const float y = ((float)(b - R) + 0.5f) / (float)u - 0.5f - yo;
        for (int a = 0; a < EW; ++a) {
          const float x = ((float)(a - R) + 0.5f) / (float)u - 0.5f - xo;
          const float xe = -x * sp + y * cp, ye = (-x * cp - y * sp) * inv_ci;
          const float r = sqrtf(xe * xe + ye * ye);
          const float cos_t = r > 0.f ? xe / r : 0.f;
          const float I = expf(-r / r0);
          const float q = r / rt;
          const float vrot = g->rc_model == 0 ? 0.63661977236758134f * vt * atanf(q) : vt * fminf(q, 1.f);
          const float vlos = vsys + vrot * si * cos_t;
          float s0 = 0.f, s1 = 0.f, s2 = 0.f;
#pragma omp simd reduction(+ : s0, s1, s2)
          for (int c = 0; c < nvx; ++c) {
            const float d = vc[c] - vlos;
            const float e = expf(d * d * inv2s2);
            s0 += w0[c] * e, s1 += w1[c] * e, s2 += w2[c] * e;
          }
          const size_t o = (size_t)b * EW + a;
          S[o] = I * s0, S[(size_t)EW * EH + o] = I * s1, S[2 * (size_t)EW * EH + o] = I * s2;
        }
      }
      /* separable PSF: x pass (EH rows x fw columns), then y pass fused with down-sampling and moments */
      for (int q = 0; q < 3; ++q)
        for (int b = 0; b < EH; ++b) {
          const float *src = S + (size_t)q * EW * EH + (size_t)b * EW;
          float *dst = T + (size_t)q * fw * EH + (size_t)b * fw;
          for (int a = 0; a < fw; ++a) dst[a] = 0.f;
          for (int j = 0; j <= 2 * R; ++j) {
            const float t = g->psf[2 * R - j];
#pragma omp simd
            for (int a = 0; a < fw; ++a) dst[a] += t * src[a + j];
          }
        }
      double acc = 0.0;
      int bad = 0;
      for (int Y = 0; Y < g->ny && !bad; ++Y)
        for (int X = 0; X < g->nx; ++X) {
          float m[3] = {0.f, 0.f, 0.f};
          for (int q = 0; q < 3; ++q) {
            const float *src = T + (size_t)q * fw * EH;
            float s = 0.f;
            for (int dy = 0; dy < u; ++dy)
              for (int j = 0; j <= 2 * R; ++j) {
                const float t = g->psf[2 * R - j];
                const float *rowp = src + (size_t)(Y * u + dy + j) * fw + X * u;
                for (int dx = 0; dx < u; ++dx) s += t * rowp[dx];
              }
            m[q] = s;
          }
          const size_t pix = (size_t)Y * g->nx + X;
          if (mask && !mask[pix]) continue;
          const float m0 = m[0] * amp * i0;
          const float m1 = m[1] / m[0], var = m[2] / m[0] - m1 * m1;
          const float m2 = sqrtf(var > 0.f ? var : 0.f);
          if (!(m0 >= 1e-30f * i0) || !isfinite(m1) || !isfinite(m2)) {
            bad = 1;
            break;
          }
          const float t = (m1 + v_ref - (vobs[pix] - g->v_center)) / verr[pix];
          const float s = sobs ? (m2 - sobs[pix]) / serr[pix] : 0.f;
          acc += (double)(t * t + s * s);
        }
      chi2[k] = bad ? INFINITY : (float)acc;
    }
    free(S);
    free(T);
    free(w);
  }
  return fail ? -1 : 0;
}
