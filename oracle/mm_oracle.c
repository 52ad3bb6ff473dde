/*
 * mm_oracle.c -- plain CPU oracle for the micromagnetic hot path of
 * arxiv/paper_2606_01114 ("Magnum.np.distributed").
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may build, load or call it.  It
 * shares no code, header, table or constant generator with the CUDA path under
 * paper_2606_01114_b200/ and neither side imports the other.
 *
 * Everything is fp64 (the Newell tensor is evaluated in __float128 and rounded once).
 * Array layout everywhere: [nx][ny][nz][3], component fastest (the
 * paper's state tensor state.m[x,y,z,c]).
 *
 * What each function follows (PAPER.md = /root/reference/PAPER.md, SURVEY = SURVEY.md):
 *   O1 orc_newell_*          Newell tensor, PAPER.md:43 (cited, not printed; ref 23) -> SURVEY 8(c) O1
 *   O2 sign/scale            PAPER.md:45 eq. 4, reading Q2: H = -Ms * sum N(r-r') m(r')
 *   O3 orc_demag_direct*     eq. 4 written out as the O(n^2) real-space sum (ground truth)
 *   O4 orc_demag_dft         the zero-padded circular convolution of PAPER.md:47 by literal DFT
 *   O5 orc_demag_fft*        the same by an own radix-2 FFT, z then y then x; period 2n,
 *                            or the next power of two above 2n when n is not one (reading Q27)
 *   O6 orc_exchange          PAPER.md:32 eq. 2, 6-point stencil, Neumann boundary (reading Q5)
 *   O7 orc_anisotropy/zeeman PAPER.md:30 (uniaxial, reading Q7), PAPER.md:140-143 (B/mu0)
 *   O8 orc_llg_rhs           PAPER.md:25 eq. 1 on unit m (reading Q4)
 *   O9 orc_rk4_step          classic RK4 + renormalise (reading Q14)
 *   O11 orc_dmi              PAPER.md:34-39 eq. 3, central differences, boundary rule of the exchange stencil (Q28)
 *   O12 orc_stt              spin-transfer torque as a local effective field a_damp (m x p) + a_field p
 *                            (PAPER.md:30 names the term; amplitudes are inputs, reading Q29)
 *   O13 orc_bb_step          Barzilai-Borwein energy minimiser iteration, PAPER.md:55, 146-148 (named only;
 *                            step rule, update and stop criterion are reading Q30)
 *   O14 orc_heff (cells)     per-cell Ms and A (eq. 2 as div(A grad M)); discrete form = reading Q31
 *   O10 orc_rkf45_step       Runge-Kutta-Fehlberg 4(5) attempt + max-error step control
 *                            (the paper names the method and the max-error reduction; tableau, error
 *                            norm and controller are readings Q23-Q26 of DESIGN.md)
 *
 * Pins: tests/test_oracle_*.py (closed forms, survey/mpmath values in tests/golden/,
 * Gauss-Legendre quadrature of the defining integral, direct-sum vs DFT vs FFT, invariants).
 * Parity unpinned: none of the functions; the SP4-shaped trajectory of config 2 has no
 * external truth in the container (SURVEY 8(c) last pin row) and is GPU-vs-oracle only.
 */
#define _GNU_SOURCE
#include <complex.h>
#include <math.h>
#include <quadmath.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef __float128 quad;

#define ORC_MU0 (4.0e-7 * M_PI) /* reading Q8: 4 pi 1e-7 T m / A */

enum { ORC_TERM_DEMAG = 1, ORC_TERM_EXCHANGE = 2, ORC_TERM_ANISOTROPY = 4, ORC_TERM_ZEEMAN = 8,
       ORC_TERM_DMI = 16, ORC_TERM_STT = 32 };

int orc_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

/* ------------------------------------------------------------------ O1: Newell f, g */

/* f(x,y,z), even in every argument.  A term whose prefactor or denominator is 0 is dropped. */
static quad newell_f(quad x, quad y, quad z) {
  x = fabsq(x); y = fabsq(y); z = fabsq(z);
  const quad x2 = x * x, y2 = y * y, z2 = z * z;
  const quad R = sqrtq(x2 + y2 + z2);
  quad r = 0;
  if (y > 0 && (x2 + z2) > 0) r += (y / 2) * (z2 - x2) * asinhq(y / sqrtq(x2 + z2));
  if (z > 0 && (x2 + y2) > 0) r += (z / 2) * (y2 - x2) * asinhq(z / sqrtq(x2 + y2));
  if (x > 0 && y > 0 && z > 0) r -= x * y * z * atanq(y * z / (x * R));
  r += (2 * x2 - y2 - z2) * R / 6;
  return r;
}

/* g(x,y,z), odd in x, odd in y, even in z. */
static quad newell_g(quad x, quad y, quad z) {
  const quad sgn = ((x < 0) ? -1 : 1) * ((y < 0) ? -1 : 1);
  x = fabsq(x); y = fabsq(y); z = fabsq(z);
  const quad x2 = x * x, y2 = y * y, z2 = z * z;
  const quad R = sqrtq(x2 + y2 + z2);
  quad r = 0;
  if (x > 0 && y > 0) {
    if (z > 0) r += x * y * z * asinhq(z / sqrtq(x2 + y2));
    r += (y / 6) * (3 * z2 - y2) * asinhq(x / sqrtq(y2 + z2));
    r += (x / 6) * (3 * z2 - x2) * asinhq(y / sqrtq(x2 + z2));
    if (z > 0) {
      r -= (z * z2 / 6) * atanq(x * y / (z * R));
      r -= (z * y2 / 2) * atanq(x * z / (y * R));
      r -= (z * x2 / 2) * atanq(y * z / (x * R));
    }
    r -= x * y * R / 3;
  }
  return sgn * r;
}

/* The six generating functions with their argument permutations:
 * xx f(x,y,z)  yy f(y,z,x)  zz f(z,x,y)  xy g(x,y,z)  xz g(x,z,y)  yz g(y,z,x) */
static quad newell_F(int comp, quad X, quad Y, quad Z) {
  switch (comp) {
    case 0: return newell_f(X, Y, Z);
    case 1: return newell_f(Y, Z, X);
    case 2: return newell_f(Z, X, Y);
    case 3: return newell_g(X, Y, Z);
    case 4: return newell_g(X, Z, Y);
    default: return newell_g(Y, Z, X);
  }
}

static int structurally_zero(int comp, int i, int j, int k) {
  if (comp == 3) return i == 0 || j == 0;
  if (comp == 4) return i == 0 || k == 0;
  if (comp == 5) return j == 0 || k == 0;
  return 0;
}

/* Literal definition at one offset: N = -D[F](X,Y,Z)/(4 pi V), D the 27-point
 * second-difference with weights (1,-2,1)^3.  out[6] = xx yy zz xy xz yz. */
void orc_newell_point(double dx, double dy, double dz, int i, int j, int k, double out[6]) {
  const quad qx = dx, qy = dy, qz = dz;
  const quad pref = -1 / (4 * M_PIq * qx * qy * qz);
  static const int w[3] = {1, -2, 1};
  for (int comp = 0; comp < 6; ++comp) {
    if (structurally_zero(comp, i, j, k)) { out[comp] = 0.0; continue; }
    quad s = 0;
    for (int a = -1; a <= 1; ++a)
      for (int b = -1; b <= 1; ++b)
        for (int c = -1; c <= 1; ++c)
          s += (quad)(w[a + 1] * w[b + 1] * w[c + 1]) *
               newell_F(comp, (i + a) * qx, (j + b) * qy, (k + c) * qz);
    out[comp] = (double)(pref * s);
  }
}

/* Octant table N[comp][i][j][k], i<nx, j<ny, k<nz, comp in xx yy zz xy xz yz.
 * Same definition; F is evaluated once per lattice point (-1..n) and D applied to the
 * stored quad values (the 27-term sum regrouped, still in quad; rounded to fp64 once). */
int orc_newell_octant(int nx, int ny, int nz, double dx, double dy, double dz, double *N) {
  if (nx < 1 || ny < 1 || nz < 1 || !(dx > 0) || !(dy > 0) || !(dz > 0) || !N) return 1;
  const size_t sx = (size_t)nx + 2, sy = (size_t)ny + 2, sz = (size_t)nz + 2;
  quad *F = (quad *)malloc(sx * sy * sz * sizeof(quad));
  if (!F) return 2;
  const quad qx = dx, qy = dy, qz = dz;
  const quad pref = -1 / (4 * M_PIq * qx * qy * qz);
  static const int w[3] = {1, -2, 1};
  for (int comp = 0; comp < 6; ++comp) {
#pragma omp parallel for collapse(2) schedule(dynamic, 4)
    for (int i = -1; i <= nx; ++i)
      for (int j = -1; j <= ny; ++j)
        for (int k = -1; k <= nz; ++k)
          F[((size_t)(i + 1) * sy + (size_t)(j + 1)) * sz + (size_t)(k + 1)] =
              newell_F(comp, i * qx, j * qy, k * qz);
#pragma omp parallel for collapse(2) schedule(static)
    for (int i = 0; i < nx; ++i)
      for (int j = 0; j < ny; ++j)
        for (int k = 0; k < nz; ++k) {
          double v = 0.0;
          if (!structurally_zero(comp, i, j, k)) {
            quad s = 0;
            for (int a = 0; a < 3; ++a)
              for (int b = 0; b < 3; ++b)
                for (int c = 0; c < 3; ++c)
                  s += (quad)(w[a] * w[b] * w[c]) *
                       F[((size_t)(i + a) * sy + (size_t)(j + b)) * sz + (size_t)(k + c)];
            v = (double)(pref * s);
          }
          N[(((size_t)comp * nx + i) * ny + j) * nz + k] = v;
        }
  }
  free(F);
  return 0;
}

/* N_rc at a signed offset from the octant table: diagonal even, xy odd in x,y, etc. */
static const int COMP_OF[3][3] = {{0, 3, 4}, {3, 1, 5}, {4, 5, 2}};

static inline double newell_lookup(const double *N, int nx, int ny, int nz, int r, int c, int di,
                                   int dj, int dk) {
  const int comp = COMP_OF[r][c];
  const int ai = di < 0 ? -di : di, aj = dj < 0 ? -dj : dj, ak = dk < 0 ? -dk : dk;
  double v = N[(((size_t)comp * nx + ai) * ny + aj) * nz + ak];
  int flip = 0;
  if (comp == 3) flip = (di < 0) ^ (dj < 0);
  if (comp == 4) flip = (di < 0) ^ (dk < 0);
  if (comp == 5) flip = (dj < 0) ^ (dk < 0);
  return flip ? -v : v;
}

/* ------------------------------------------------------------------ O3: direct sum */

static void direct_at(int nx, int ny, int nz, const double *N, double Ms, const double *m, int xi,
                      int yi, int zi, double out[3]) {
  long double acc[3] = {0, 0, 0};
  for (int x = 0; x < nx; ++x)
    for (int y = 0; y < ny; ++y)
      for (int z = 0; z < nz; ++z) {
        const double *mj = m + (((size_t)x * ny + y) * nz + z) * 3;
        for (int r = 0; r < 3; ++r)
          for (int c = 0; c < 3; ++c)
            acc[r] += (long double)newell_lookup(N, nx, ny, nz, r, c, xi - x, yi - y, zi - z) *
                      (long double)mj[c];
      }
  for (int r = 0; r < 3; ++r) out[r] = (double)(-(long double)Ms * acc[r]);
}

/* H(i) = -Ms sum_j N(i-j) m(j) for every cell (O(n^2)). */
int orc_demag_direct(int nx, int ny, int nz, const double *N, double Ms, const double *m,
                     double *H) {
#pragma omp parallel for collapse(2) schedule(dynamic, 1)
  for (int x = 0; x < nx; ++x)
    for (int y = 0; y < ny; ++y)
      for (int z = 0; z < nz; ++z)
        direct_at(nx, ny, nz, N, Ms, m, x, y, z, H + (((size_t)x * ny + y) * nz + z) * 3);
  return 0;
}

/* The same sum at nsamp chosen cells (flat cell index (x*ny+y)*nz+z); Hs[nsamp][3]. */
int orc_demag_direct_sampled(int nx, int ny, int nz, const double *N, double Ms, const double *m,
                             int nsamp, const int64_t *cells, double *Hs) {
#pragma omp parallel for schedule(dynamic, 1)
  for (int s = 0; s < nsamp; ++s) {
    const int64_t c = cells[s];
    const int z = (int)(c % nz), y = (int)((c / nz) % ny), x = (int)(c / ((int64_t)nz * ny));
    direct_at(nx, ny, nz, N, Ms, m, x, y, z, Hs + (size_t)s * 3);
  }
  return 0;
}

/* ------------------------------------------------------------------ padded grids */

static int padded(int n) { return n == 1 ? 1 : 2 * n; } /* reading Q10 */

/* Mirror the octant table onto the padded (periodic) grid of period Px x Py x Pz >= 2n (or 1):
 * offset -i sits at index P-i, the unused indices (distance >= n, never needed) are 0
 * (reading Q11).  out[Px][Py][Pz] for one component. */
static void mirror_fill(const double *N, int nx, int ny, int nz, int Px, int Py, int Pz, int comp,
                        double complex *out) {
  for (int a = 0; a < Px; ++a)
    for (int b = 0; b < Py; ++b)
      for (int c = 0; c < Pz; ++c) {
        const int di = a < nx ? a : a - Px, dj = b < ny ? b : b - Py, dk = c < nz ? c : c - Pz;
        double v = 0.0;
        /* offsets of magnitude >= n never occur between two cells of the mesh: 0 (for P = 2n
         * that is the single index n; for a longer period the whole gap n .. P-n) */
        if (abs(di) < nx && abs(dj) < ny && abs(dk) < nz) {
          const int r = comp < 3 ? comp : (comp == 5 ? 1 : 0);
          const int cc = comp < 3 ? comp : (comp == 3 ? 1 : 2);
          v = newell_lookup(N, nx, ny, nz, r, cc, di, dj, dk);
        }
        out[((size_t)a * Py + b) * Pz + c] = v;
      }
}

/* ------------------------------------------------------------------ O4: literal DFT */

/* Zero-padded circular convolution by literal 3D DFTs (no FFT algorithm at all).
 * Only for tiny meshes: cost ~ 9 * (Px Py Pz)^2. */
int orc_demag_dft(int nx, int ny, int nz, const double *N, double Ms, const double *m, double *H) {
  const int Px = padded(nx), Py = padded(ny), Pz = padded(nz);
  const size_t P = (size_t)Px * Py * Pz;
  if (P > 8192) return 3;
  double complex *Nr = malloc(6 * P * sizeof(double complex));
  double complex *Nk = malloc(6 * P * sizeof(double complex));
  double complex *mr = calloc(3 * P, sizeof(double complex));
  double complex *mk = malloc(3 * P * sizeof(double complex));
  double complex *hk = malloc(3 * P * sizeof(double complex));
  if (!Nr || !Nk || !mr || !mk || !hk) return 2;
  for (int comp = 0; comp < 6; ++comp) mirror_fill(N, nx, ny, nz, Px, Py, Pz, comp, Nr + comp * P);
  for (int x = 0; x < nx; ++x)
    for (int y = 0; y < ny; ++y)
      for (int z = 0; z < nz; ++z)
        for (int c = 0; c < 3; ++c)
          mr[c * P + ((size_t)x * Py + y) * Pz + z] = m[(((size_t)x * ny + y) * nz + z) * 3 + c];
  /* forward: X(k) = sum_r x(r) exp(-2 pi i (kx rx/Px + ky ry/Py + kz rz/Pz)) */
#pragma omp parallel for schedule(static)
  for (long kk = 0; kk < (long)P; ++kk) {
    const int kx = (int)(kk / ((long)Py * Pz)), ky = (int)((kk / Pz) % Py), kz = (int)(kk % Pz);
    double complex accN[6] = {0}, accm[3] = {0};
    for (int a = 0; a < Px; ++a)
      for (int b = 0; b < Py; ++b)
        for (int c = 0; c < Pz; ++c) {
          const double ph = -2.0 * M_PI *
                            ((double)((long)kx * a % Px) / Px + (double)((long)ky * b % Py) / Py +
                             (double)((long)kz * c % Pz) / Pz);
          const double complex w = cos(ph) + I * sin(ph);
          const size_t r = ((size_t)a * Py + b) * Pz + c;
          for (int q = 0; q < 6; ++q) accN[q] += Nr[q * P + r] * w;
          for (int q = 0; q < 3; ++q) accm[q] += mr[q * P + r] * w;
        }
    for (int q = 0; q < 6; ++q) Nk[q * P + kk] = accN[q];
    for (int q = 0; q < 3; ++q) mk[q * P + kk] = accm[q];
  }
  for (size_t kk = 0; kk < P; ++kk)
    for (int r = 0; r < 3; ++r) {
      double complex s = 0;
      for (int c = 0; c < 3; ++c) s += Nk[COMP_OF[r][c] * P + kk] * mk[c * P + kk];
      hk[r * P + kk] = s;
    }
  /* inverse at the physical cells only, 1/P normalisation, times -Ms (O2) */
#pragma omp parallel for collapse(2) schedule(static)
  for (int x = 0; x < nx; ++x)
    for (int y = 0; y < ny; ++y)
      for (int z = 0; z < nz; ++z) {
        double complex acc[3] = {0};
        for (int a = 0; a < Px; ++a)
          for (int b = 0; b < Py; ++b)
            for (int c = 0; c < Pz; ++c) {
              const double ph = 2.0 * M_PI *
                                ((double)((long)a * x % Px) / Px + (double)((long)b * y % Py) / Py +
                                 (double)((long)c * z % Pz) / Pz);
              const double complex w = cos(ph) + I * sin(ph);
              const size_t k = ((size_t)a * Py + b) * Pz + c;
              for (int r = 0; r < 3; ++r) acc[r] += hk[r * P + k] * w;
            }
        for (int r = 0; r < 3; ++r)
          H[(((size_t)x * ny + y) * nz + z) * 3 + r] = -Ms * creal(acc[r]) / (double)P;
      }
  free(Nr); free(Nk); free(mr); free(mk); free(hk);
  return 0;
}

/* ------------------------------------------------------------------ O5: own FFT path */

/* Period of the FFT path along an axis of n cells: 2n when n is a power of two (the paper's
 * zero-padding), else the next power of two above 2n.  A circular convolution of
 * any period P >= 2n - 1 equals the linear convolution of eq. 4 on the n cells (the wrapped
 * images fall on zero padding), so the field does not depend on this choice (DESIGN.md reading
 * Q27); it keeps the oracle's FFT the textbook radix-2 one.  orc_fft_period exports it. */
int orc_fft_period(int n) {
  if (n == 1) return 1;
  int P = 2;
  while (P < 2 * n) P *= 2;
  return P;
}

/* Textbook iterative radix-2 decimation-in-time FFT on a contiguous buffer of length n
 * (power of two).  sign = -1 forward, +1 inverse (unnormalised).  tw[q] = exp(sign 2 pi i q/n). */
static void fft_radix2(double complex *a, int n, const double complex *tw) {
  for (int i = 1, j = 0; i < n; ++i) { /* bit reversal */
    int bit = n >> 1;
    for (; j & bit; bit >>= 1) j ^= bit;
    j ^= bit;
    if (i < j) { double complex t = a[i]; a[i] = a[j]; a[j] = t; }
  }
  for (int len = 2; len <= n; len <<= 1) {
    const int half = len >> 1, step = n / len;
    for (int s = 0; s < n; s += len)
      for (int q = 0; q < half; ++q) {
        const double complex u = a[s + q], v = a[s + q + half] * tw[q * step];
        a[s + q] = u + v;
        a[s + q + half] = u - v;
      }
  }
}

static double complex *make_twiddles(int n, int sign) {
  double complex *tw = malloc((size_t)(n > 0 ? n : 1) * sizeof(double complex));
  for (int q = 0; q < n; ++q) {
    const double ph = sign * 2.0 * M_PI * (double)q / (double)n;
    tw[q] = cos(ph) + I * sin(ph);
  }
  return tw;
}

/* 1D FFTs along one axis of a [Px][Py][Pz] complex array, for index ranges
 * x<limx, y<limy, z<limz of the *other* axes (pencils outside are known zero / unneeded). */
static void fft_axis(double complex *A, int Px, int Py, int Pz, int axis, int sign, int lim0,
                     int lim1) {
  const int n = axis == 0 ? Px : (axis == 1 ? Py : Pz);
  if (n == 1) return;
  double complex *tw = make_twiddles(n, sign);
#pragma omp parallel
  {
    double complex *buf = malloc((size_t)n * sizeof(double complex));
#pragma omp for collapse(2) schedule(static)
    for (int p = 0; p < lim0; ++p)
      for (int q = 0; q < lim1; ++q) {
        size_t base, stride;
        if (axis == 2) { base = ((size_t)p * Py + q) * Pz; stride = 1; }            /* (x,y) */
        else if (axis == 1) { base = (size_t)p * Py * Pz + q; stride = Pz; }       /* (x,z) */
        else { base = (size_t)p * Pz + q; stride = (size_t)Py * Pz; }             /* (y,z) */
        for (int t = 0; t < n; ++t) buf[t] = A[base + t * stride];
        fft_radix2(buf, n, tw);
        for (int t = 0; t < n; ++t) A[base + t * stride] = buf[t];
      }
    free(buf);
  }
  free(tw);
}

/* Fourier-space tensor: real part of the forward 3D FFT of the mirrored table,
 * Nhat[6][Px][Py][Pz] (the imaginary part is analytically zero; its measured max is
 * returned through max_imag if non-NULL). */
int orc_demag_fft_nhat(int nx, int ny, int nz, const double *N, double *Nhat, double *max_imag) {
  const int Px = orc_fft_period(nx), Py = orc_fft_period(ny), Pz = orc_fft_period(nz);
  const size_t P = (size_t)Px * Py * Pz;
  double complex *A = malloc(P * sizeof(double complex));
  if (!A) return 2;
  double mi = 0.0;
  for (int comp = 0; comp < 6; ++comp) {
    mirror_fill(N, nx, ny, nz, Px, Py, Pz, comp, A);
    fft_axis(A, Px, Py, Pz, 2, -1, Px, Py);
    fft_axis(A, Px, Py, Pz, 1, -1, Px, Pz);
    fft_axis(A, Px, Py, Pz, 0, -1, Py, Pz);
    for (size_t k = 0; k < P; ++k) {
      Nhat[comp * P + k] = creal(A[k]);
      if (fabs(cimag(A[k])) > mi) mi = fabs(cimag(A[k]));
    }
  }
  if (max_imag) *max_imag = mi;
  free(A);
  return 0;
}

/* H = -Ms * crop( IFFT( Nhat . FFT( pad(m) ) ) ), z then y then x forward,
 * x then y then z inverse.  Pencils that are all zero (forward) or whose outputs are
 * discarded (inverse) are skipped; that changes no value. */
int orc_demag_fft(int nx, int ny, int nz, const double *Nhat, double Ms, const double *m,
                  double *H) {
  const int Px = orc_fft_period(nx), Py = orc_fft_period(ny), Pz = orc_fft_period(nz);
  const size_t P = (size_t)Px * Py * Pz;
  double complex *A = calloc(3 * P, sizeof(double complex));
  if (!A) return 2;
  for (int c = 0; c < 3; ++c) {
    double complex *Ac = A + c * P;
#pragma omp parallel for collapse(2) schedule(static)
    for (int x = 0; x < nx; ++x)
      for (int y = 0; y < ny; ++y)
        for (int z = 0; z < nz; ++z)
          Ac[((size_t)x * Py + y) * Pz + z] = m[(((size_t)x * ny + y) * nz + z) * 3 + c];
    fft_axis(Ac, Px, Py, Pz, 2, -1, nx, ny);
    fft_axis(Ac, Px, Py, Pz, 1, -1, nx, Pz);
    fft_axis(Ac, Px, Py, Pz, 0, -1, Py, Pz);
  }
#pragma omp parallel for schedule(static)
  for (long k = 0; k < (long)P; ++k) {
    double complex mk[3] = {A[k], A[P + k], A[2 * P + k]}, hk[3];
    for (int r = 0; r < 3; ++r) {
      hk[r] = 0;
      for (int c = 0; c < 3; ++c) hk[r] += Nhat[COMP_OF[r][c] * P + k] * mk[c];
    }
    for (int r = 0; r < 3; ++r) A[r * P + k] = hk[r];
  }
  for (int c = 0; c < 3; ++c) {
    double complex *Ac = A + c * P;
    fft_axis(Ac, Px, Py, Pz, 0, +1, Py, Pz);
    fft_axis(Ac, Px, Py, Pz, 1, +1, nx, Pz);
    fft_axis(Ac, Px, Py, Pz, 2, +1, nx, ny);
#pragma omp parallel for collapse(2) schedule(static)
    for (int x = 0; x < nx; ++x)
      for (int y = 0; y < ny; ++y)
        for (int z = 0; z < nz; ++z)
          H[(((size_t)x * ny + y) * nz + z) * 3 + c] =
              -Ms * creal(Ac[((size_t)x * Py + y) * Pz + z]) / (double)P;
  }
  free(A);
  return 0;
}

/* ------------------------------------------------------------------ O6, O7 local terms */

/* H_ex = 2A/(mu0 Ms) sum_d [m(i+e_d) - 2 m(i) + m(i-e_d)] / D_d^2; a neighbour outside
 * the mesh is replaced by m(i) (Neumann), so an axis with n_d = 1 contributes 0. */
int orc_exchange(int nx, int ny, int nz, double dx, double dy, double dz, double Ms, double Aex,
                 const double *m, double *H) {
  const double pref = 2.0 * Aex / (ORC_MU0 * Ms);
  const double inv[3] = {1.0 / (dx * dx), 1.0 / (dy * dy), 1.0 / (dz * dz)};
  const int n[3] = {nx, ny, nz};
#pragma omp parallel for collapse(2) schedule(static)
  for (int x = 0; x < nx; ++x)
    for (int y = 0; y < ny; ++y)
      for (int z = 0; z < nz; ++z) {
        const int idx[3] = {x, y, z};
        const size_t i0 = (((size_t)x * ny + y) * nz + z) * 3;
        for (int c = 0; c < 3; ++c) {
          double lap = 0.0;
          for (int d = 0; d < 3; ++d) {
            int ip[3] = {x, y, z}, im[3] = {x, y, z};
            ip[d] = idx[d] + 1 < n[d] ? idx[d] + 1 : idx[d];
            im[d] = idx[d] - 1 >= 0 ? idx[d] - 1 : idx[d];
            const double mp = m[(((size_t)ip[0] * ny + ip[1]) * nz + ip[2]) * 3 + c];
            const double mm = m[(((size_t)im[0] * ny + im[1]) * nz + im[2]) * 3 + c];
            lap += (mp - 2.0 * m[i0 + c] + mm) * inv[d];
          }
          H[i0 + c] = pref * lap;
        }
      }
  return 0;
}

/* H_an = 2Ku/(mu0 Ms) (m.u) u, u a unit vector. */
int orc_anisotropy(size_t ncell, double Ms, double Ku, const double u[3], const double *m,
                   double *H) {
  const double pref = 2.0 * Ku / (ORC_MU0 * Ms);
  for (size_t i = 0; i < ncell; ++i) {
    const double d = m[3 * i] * u[0] + m[3 * i + 1] * u[1] + m[3 * i + 2] * u[2];
    for (int c = 0; c < 3; ++c) H[3 * i + c] = pref * d * u[c];
  }
  return 0;
}

/* O11 DMI (eq. 3): H = 2D/(mu0 Ms) sum_{k=x,y,z} e_k^DMI x dm/dk, with the three
 * DMI vectors e_k^DMI given as e[k][0..2] (interfacial: e_x = (0,1,0), e_y = (-1,0,0), e_z = 0;
 * bulk: e_k = unit vector k).  dm/dk is the central difference
 * (m(i+e_k) - m(i-e_k)) / (2 D_k); a neighbour outside the mesh is replaced by the cell itself
 * (the rule of the exchange stencil, reading Q5; reading Q28), so an axis with
 * n_k = 1 contributes 0. */
int orc_dmi(int nx, int ny, int nz, double dx, double dy, double dz, double Ms, double D,
            const double e[9], const double *m, double *H) {
  const double pref = 2.0 * D / (ORC_MU0 * Ms);
  const double h[3] = {dx, dy, dz};
  const int n[3] = {nx, ny, nz};
#pragma omp parallel for collapse(2) schedule(static)
  for (int x = 0; x < nx; ++x)
    for (int y = 0; y < ny; ++y)
      for (int z = 0; z < nz; ++z) {
        const int idx[3] = {x, y, z};
        const size_t i0 = (((size_t)x * ny + y) * nz + z) * 3;
        double acc[3] = {0, 0, 0};
        for (int k = 0; k < 3; ++k) {
          int ip[3] = {x, y, z}, im[3] = {x, y, z};
          ip[k] = idx[k] + 1 < n[k] ? idx[k] + 1 : idx[k];
          im[k] = idx[k] - 1 >= 0 ? idx[k] - 1 : idx[k];
          double dm[3];
          for (int c = 0; c < 3; ++c)
            dm[c] = (m[(((size_t)ip[0] * ny + ip[1]) * nz + ip[2]) * 3 + c] -
                     m[(((size_t)im[0] * ny + im[1]) * nz + im[2]) * 3 + c]) / (2.0 * h[k]);
          const double *ek = e + 3 * k;
          acc[0] += ek[1] * dm[2] - ek[2] * dm[1];
          acc[1] += ek[2] * dm[0] - ek[0] * dm[2];
          acc[2] += ek[0] * dm[1] - ek[1] * dm[0];
        }
        for (int c = 0; c < 3; ++c) H[i0 + c] = pref * acc[c];
      }
  return 0;
}

/* O12 spin-transfer torque as an effective field (PAPER.md:30 names the Slonczewski torque as a
 * local term; its prefactors are not printed): H = a_damp (m x p) + a_field p with a unit
 * polarisation p and the two amplitudes in A/m given by the caller (reading Q29).
 * Under eq. 1 the first part gives the damping-like torque ~ m x (m x p), the second the
 * field-like torque ~ m x p. */
int orc_stt(size_t ncell, const double pvec[3], double a_damp, double a_field, const double *m, double *H) {
  for (size_t i = 0; i < ncell; ++i) {
    const double *mi = m + 3 * i;
    H[3 * i + 0] = a_damp * (mi[1] * pvec[2] - mi[2] * pvec[1]) + a_field * pvec[0];
    H[3 * i + 1] = a_damp * (mi[2] * pvec[0] - mi[0] * pvec[2]) + a_field * pvec[1];
    H[3 * i + 2] = a_damp * (mi[0] * pvec[1] - mi[1] * pvec[0]) + a_field * pvec[2];
  }
  return 0;
}

/* ------------------------------------------------------------------ problem + O8, O9 */

typedef struct {
  int nx, ny, nz;
  double dx, dy, dz;
  double Ms, Aex, Ku, axis[3], alpha, gamma, Hext[3];
  unsigned terms;
  const double *Nhat; /* from orc_demag_fft_nhat; required if DEMAG is enabled */
  double D, edmi[9];                      /* DMI constant (J/m^2) and the three DMI vectors */
  double stt_p[3], stt_damp, stt_field;   /* spin-torque field: unit polarisation, amplitudes (A/m) */
  const double *Ms_cells, *A_cells;       /* per-cell Ms (A/m) and A (J/m), [nx][ny][nz]; NULL = uniform Ms / Aex */
} orc_problem;

/* O14 inhomogeneous material parameters ("inhomogeneous material parameters"; eq. 2 is
 * written as div(A grad M) for that reason; the discrete form is DESIGN.md reading Q31):
 *   demag     H(i) = - sum_j N(i - j) Ms_j m_j                                   (M = Ms m, eq. 4)
 *   exchange  H(i) = 2/(mu0 Ms_i) sum_{d, +-} A_ij (m_j - m_i) / D_d^2,  A_ij = 2 A_i A_j / (A_i + A_j)
 *             (harmonic mean: the flux A dm/dx is continuous across the interface; 0 if either is 0),
 *             a neighbour outside the mesh or in vacuum (Ms_j = 0) contributes nothing (Q5)
 *   anisotropy, DMI: the homogeneous formulas with Ms_i; for DMI a neighbour with Ms_j = 0 counts as
 *             outside the mesh (replaced by the cell itself, Q28)
 *   a cell with Ms_i = 0 is vacuum: the terms with a 1/Ms_i prefactor vanish there and dm/dt = 0.
 * Ms_i(p, i), A_i(p, i) read the arrays or fall back to the uniform values. */
static double ms_at(const orc_problem *p, size_t i) { return p->Ms_cells ? p->Ms_cells[i] : p->Ms; }
static double a_at(const orc_problem *p, size_t i) { return p->A_cells ? p->A_cells[i] : p->Aex; }

static int orc_heff_cells(const orc_problem *p, const double *m, double *H) {
  const int nx = p->nx, ny = p->ny, nz = p->nz;
  const size_t n = (size_t)nx * ny * nz;
  const double h[3] = {p->dx, p->dy, p->dz};
  const int nn[3] = {nx, ny, nz};
  memset(H, 0, 3 * n * sizeof(double));
  if (p->terms & ORC_TERM_DEMAG) {
    if (!p->Nhat) return 3;
    double *Mm = malloc(3 * n * sizeof(double)), *T = malloc(3 * n * sizeof(double));
    if (!Mm || !T) { free(Mm); free(T); return 2; }
    for (size_t i = 0; i < n; ++i)
      for (int c = 0; c < 3; ++c) Mm[3 * i + c] = ms_at(p, i) * m[3 * i + c];
    int rc = orc_demag_fft(nx, ny, nz, p->Nhat, 1.0, Mm, T);   /* - sum N M */
    if (!rc) for (size_t i = 0; i < 3 * n; ++i) H[i] += T[i];
    free(Mm); free(T);
    if (rc) return rc;
  }
#pragma omp parallel for collapse(2) schedule(static)
  for (int x = 0; x < nx; ++x)
    for (int y = 0; y < ny; ++y)
      for (int z = 0; z < nz; ++z) {
        const int idx[3] = {x, y, z};
        const size_t ci = ((size_t)x * ny + y) * nz + z, i0 = 3 * ci;
        const double Msi = ms_at(p, ci), Ai = a_at(p, ci);
        double acc[3] = {0, 0, 0};
        if (Msi > 0.0) {
          for (int d = 0; d < 3; ++d) {
            double dm[3] = {0, 0, 0};   /* m(+) - m(-) with the boundary / vacuum rule, for DMI */
            for (int sgn = -1; sgn <= 1; sgn += 2) {
              int j[3] = {x, y, z};
              j[d] += sgn;
              const int inside = j[d] >= 0 && j[d] < nn[d];
              const size_t cj = inside ? ((size_t)j[0] * ny + j[1]) * nz + j[2] : ci;
              const double Msj = ms_at(p, cj), Aj = a_at(p, cj);
              /* a vacuum neighbour (Ms_j = 0) is outside the magnet: no exchange partner, whatever
               * A_j and the frozen m_j stored there are (reading Q31: interface = mesh boundary) */
              if ((p->terms & ORC_TERM_EXCHANGE) && inside && Msj > 0.0 && Ai + Aj > 0.0) {
                const double Aij = 2.0 * Ai * Aj / (Ai + Aj);
                for (int c = 0; c < 3; ++c)
                  acc[c] += 2.0 / (ORC_MU0 * Msi) * Aij * (m[3 * cj + c] - m[i0 + c]) / (h[d] * h[d]);
              }
              const size_t cd = (inside && Msj > 0.0) ? cj : ci;
              for (int c = 0; c < 3; ++c) dm[c] += sgn * m[3 * cd + c];
            }
            if (p->terms & ORC_TERM_DMI) {
              const double *ek = p->edmi + 3 * d;
              const double f = 2.0 * p->D / (ORC_MU0 * Msi) / (2.0 * h[d]);
              acc[0] += f * (ek[1] * dm[2] - ek[2] * dm[1]);
              acc[1] += f * (ek[2] * dm[0] - ek[0] * dm[2]);
              acc[2] += f * (ek[0] * dm[1] - ek[1] * dm[0]);
            }
          }
          if (p->terms & ORC_TERM_ANISOTROPY) {
            const double dot = m[i0] * p->axis[0] + m[i0 + 1] * p->axis[1] + m[i0 + 2] * p->axis[2];
            for (int c = 0; c < 3; ++c) acc[c] += 2.0 * p->Ku / (ORC_MU0 * Msi) * dot * p->axis[c];
          }
        }
        if (p->terms & ORC_TERM_ZEEMAN)
          for (int c = 0; c < 3; ++c) acc[c] += p->Hext[c];
        if (p->terms & ORC_TERM_STT) {
          const double *mi = m + i0, *pv = p->stt_p;
          acc[0] += p->stt_damp * (mi[1] * pv[2] - mi[2] * pv[1]) + p->stt_field * pv[0];
          acc[1] += p->stt_damp * (mi[2] * pv[0] - mi[0] * pv[2]) + p->stt_field * pv[1];
          acc[2] += p->stt_damp * (mi[0] * pv[1] - mi[1] * pv[0]) + p->stt_field * pv[2];
        }
        for (int c = 0; c < 3; ++c) H[i0 + c] += acc[c];
      }
  return 0;
}

/* H_eff = sum of enabled terms. */
int orc_heff(const orc_problem *p, const double *m, double *H) {
  if (p->Ms_cells || p->A_cells) return orc_heff_cells(p, m, H);
  const size_t n = (size_t)p->nx * p->ny * p->nz;
  double *T = malloc(3 * n * sizeof(double));
  if (!T) return 2;
  memset(H, 0, 3 * n * sizeof(double));
  if (p->terms & ORC_TERM_DEMAG) {
    if (!p->Nhat) { free(T); return 3; }
    int rc = orc_demag_fft(p->nx, p->ny, p->nz, p->Nhat, p->Ms, m, T);
    if (rc) { free(T); return rc; }
    for (size_t i = 0; i < 3 * n; ++i) H[i] += T[i];
  }
  if (p->terms & ORC_TERM_EXCHANGE) {
    orc_exchange(p->nx, p->ny, p->nz, p->dx, p->dy, p->dz, p->Ms, p->Aex, m, T);
    for (size_t i = 0; i < 3 * n; ++i) H[i] += T[i];
  }
  if (p->terms & ORC_TERM_ANISOTROPY) {
    orc_anisotropy(n, p->Ms, p->Ku, p->axis, m, T);
    for (size_t i = 0; i < 3 * n; ++i) H[i] += T[i];
  }
  if (p->terms & ORC_TERM_ZEEMAN)
    for (size_t i = 0; i < n; ++i)
      for (int c = 0; c < 3; ++c) H[3 * i + c] += p->Hext[c];
  if (p->terms & ORC_TERM_DMI) {
    orc_dmi(p->nx, p->ny, p->nz, p->dx, p->dy, p->dz, p->Ms, p->D, p->edmi, m, T);
    for (size_t i = 0; i < 3 * n; ++i) H[i] += T[i];
  }
  if (p->terms & ORC_TERM_STT) {
    orc_stt(n, p->stt_p, p->stt_damp, p->stt_field, m, T);
    for (size_t i = 0; i < 3 * n; ++i) H[i] += T[i];
  }
  free(T);
  return 0;
}

static void cross3(const double a[3], const double b[3], double o[3]) {
  o[0] = a[1] * b[2] - a[2] * b[1];
  o[1] = a[2] * b[0] - a[0] * b[2];
  o[2] = a[0] * b[1] - a[1] * b[0];
}

/* dm/dt = -gamma/(1+alpha^2) [ m x H + alpha m x (m x H) ]   (eq. 1) */
int orc_llg_torque(size_t ncell, double alpha, double gamma, const double *m, const double *H,
                   double *dmdt) {
  const double pref = -gamma / (1.0 + alpha * alpha);
  for (size_t i = 0; i < ncell; ++i) {
    double mxh[3], mxmxh[3];
    cross3(m + 3 * i, H + 3 * i, mxh);
    cross3(m + 3 * i, mxh, mxmxh);
    for (int c = 0; c < 3; ++c) dmdt[3 * i + c] = pref * (mxh[c] + alpha * mxmxh[c]);
  }
  return 0;
}

int orc_llg_rhs(const orc_problem *p, const double *m, double *dmdt) {
  const size_t n = (size_t)p->nx * p->ny * p->nz;
  double *H = malloc(3 * n * sizeof(double));
  if (!H) return 2;
  int rc = orc_heff(p, m, H);
  if (!rc) rc = orc_llg_torque(n, p->alpha, p->gamma, m, H, dmdt);
  if (!rc && p->Ms_cells)   /* vacuum cells (Ms_i = 0) carry no magnetisation: dm/dt = 0 (O14) */
    for (size_t i = 0; i < n; ++i)
      if (!(p->Ms_cells[i] > 0.0)) dmdt[3 * i] = dmdt[3 * i + 1] = dmdt[3 * i + 2] = 0.0;
  free(H);
  return rc;
}

/* Classic RK4, then m <- m/|m| per cell; stage vectors are not renormalised. */
int orc_rk4_step(const orc_problem *p, double *m, double dt) {
  const size_t n3 = (size_t)p->nx * p->ny * p->nz * 3;
  double *k1 = malloc(4 * n3 * sizeof(double)), *ms = malloc(n3 * sizeof(double));
  if (!k1 || !ms) return 2;
  double *k2 = k1 + n3, *k3 = k2 + n3, *k4 = k3 + n3;
  int rc = orc_llg_rhs(p, m, k1);
  for (size_t i = 0; i < n3; ++i) ms[i] = m[i] + 0.5 * dt * k1[i];
  if (!rc) rc = orc_llg_rhs(p, ms, k2);
  for (size_t i = 0; i < n3; ++i) ms[i] = m[i] + 0.5 * dt * k2[i];
  if (!rc) rc = orc_llg_rhs(p, ms, k3);
  for (size_t i = 0; i < n3; ++i) ms[i] = m[i] + dt * k3[i];
  if (!rc) rc = orc_llg_rhs(p, ms, k4);
  if (!rc) {
    for (size_t i = 0; i < n3; ++i) m[i] += dt / 6.0 * (k1[i] + 2.0 * k2[i] + 2.0 * k3[i] + k4[i]);
    for (size_t i = 0; i < n3; i += 3) {
      const double nrm = sqrt(m[i] * m[i] + m[i + 1] * m[i + 1] + m[i + 2] * m[i + 2]);
      if (nrm > 0.0) { m[i] /= nrm; m[i + 1] /= nrm; m[i + 2] /= nrm; }   /* a zero vector (vacuum cell) stays zero */
    }
  }
  free(k1); free(ms);
  return rc;
}

/* O10.  One attempted step of the Runge-Kutta-Fehlberg 4(5) pair ("only the
 * Runge-Kutta-Fehlberg Method (RKF45) is supported"; "globally reduces the maximum
 * error before computing the next step size").  Fehlberg's 1969 tableau, written out:
 *   c = 0, 1/4, 3/8, 12/13, 1, 1/2
 *   k1 = f(m)
 *   k2 = f(m + dt (1/4 k1))
 *   k3 = f(m + dt (3/32 k1 + 9/32 k2))
 *   k4 = f(m + dt (1932/2197 k1 - 7200/2197 k2 + 7296/2197 k3))
 *   k5 = f(m + dt (439/216 k1 - 8 k2 + 3680/513 k3 - 845/4104 k4))
 *   k6 = f(m + dt (-8/27 k1 + 2 k2 - 3544/2565 k3 + 1859/4104 k4 - 11/40 k5))
 *   m4 = m + dt (25/216 k1 + 1408/2565 k3 + 2197/4104 k4 - 1/5 k5)
 *   m5 = m + dt (16/135 k1 + 6656/12825 k3 + 28561/56430 k4 - 9/50 k5 + 2/55 k6)
 * Readings (Q23-Q26): err = max over cells and components of |m5 - m4|, evaluated as
 * |dt sum_j (b5_j - b4_j) k_j|; the step is
 * accepted iff err <= tol; an accepted step continues with the 5th-order value, renormalised per
 * cell (m <- m5/|m5|), stage vectors are not renormalised; the next step size, after an accepted
 * and after a rejected attempt alike, is dt * min(5, max(0.2, 0.9 (tol/err)^(1/5))) clamped to
 * [dt_min, dt_max] (err = 0 -> factor 5).
 * m is updated in place only if the step is accepted.  Outputs: *err, *accepted (0/1), *dt_next. */
int orc_rkf45_step(const orc_problem *p, double *m, double dt, double tol, double dt_min,
                   double dt_max, double *err, int *accepted, double *dt_next) {
  static const double A[6][5] = {
      {0, 0, 0, 0, 0},
      {1.0 / 4.0, 0, 0, 0, 0},
      {3.0 / 32.0, 9.0 / 32.0, 0, 0, 0},
      {1932.0 / 2197.0, -7200.0 / 2197.0, 7296.0 / 2197.0, 0, 0},
      {439.0 / 216.0, -8.0, 3680.0 / 513.0, -845.0 / 4104.0, 0},
      {-8.0 / 27.0, 2.0, -3544.0 / 2565.0, 1859.0 / 4104.0, -11.0 / 40.0}};
  static const double B4[6] = {25.0 / 216.0, 0, 1408.0 / 2565.0, 2197.0 / 4104.0, -1.0 / 5.0, 0};
  static const double B5[6] = {16.0 / 135.0, 0, 6656.0 / 12825.0, 28561.0 / 56430.0, -9.0 / 50.0,
                               2.0 / 55.0};
  const size_t n3 = (size_t)p->nx * p->ny * p->nz * 3;
  double *k = malloc(6 * n3 * sizeof(double)), *ms = malloc(n3 * sizeof(double));
  if (!k || !ms) { free(k); free(ms); return 2; }
  int rc = 0;
  for (int i = 0; i < 6 && !rc; ++i) {
    for (size_t q = 0; q < n3; ++q) {
      double s = 0.0;
      for (int j = 0; j < i; ++j) s += A[i][j] * k[(size_t)j * n3 + q];
      ms[q] = m[q] + dt * s;
    }
    rc = orc_llg_rhs(p, ms, k + (size_t)i * n3);
  }
  if (!rc) {
    double e = 0.0;
    for (size_t q = 0; q < n3; ++q) {
      double s5 = 0.0, sd = 0.0;
      for (int j = 0; j < 6; ++j) {
        s5 += B5[j] * k[(size_t)j * n3 + q];
        sd += (B5[j] - B4[j]) * k[(size_t)j * n3 + q];
      }
      ms[q] = m[q] + dt * s5;
      /* m5 - m4 = dt sum_j (b5_j - b4_j) k_j, taken before the two O(1) states are formed so
       * that the estimate (1e-6 .. 1e-12) is not rounded at 1e-16 absolute (reading Q24) */
      const double d = fabs(dt * sd);
      if (d > e) e = d;
    }
    *err = e;
    *accepted = e <= tol ? 1 : 0;
    double fac = e > 0.0 ? 0.9 * pow(tol / e, 0.2) : 5.0;
    if (fac > 5.0) fac = 5.0;
    if (fac < 0.2) fac = 0.2;
    double dn = dt * fac;
    if (dn < dt_min) dn = dt_min;
    if (dn > dt_max) dn = dt_max;
    *dt_next = dn;
    if (*accepted) {
      for (size_t q = 0; q < n3; q += 3) {
        const double nrm = sqrt(ms[q] * ms[q] + ms[q + 1] * ms[q + 1] + ms[q + 2] * ms[q + 2]);
        if (nrm > 0.0) { m[q] = ms[q] / nrm; m[q + 1] = ms[q + 1] / nrm; m[q + 2] = ms[q + 2] / nrm; }
      }
    }
  }
  free(k); free(ms);
  return rc;
}

/* O13.  One iteration of the Barzilai-Borwein energy minimiser ("The
 * Barzikai-Borwein algorithm for minimising the system energy ... all ranks terminate together
 * after the convergence criteria are met"; PAPER.md:146-148 minimizer.minimize(state)).  The
 * paper names the algorithm only; the scheme is DESIGN.md reading Q30 (steepest descent on the
 * unit sphere with Barzilai-Borwein step lengths and a norm-preserving update):
 *   H_n = H_eff(m_n),   g_n = m_n x (m_n x H_n)            (the tangential energy gradient, A/m)
 *   n = 0:  tau = tau0
 *   n > 0:  s = m_n - m_{n-1},  y = g_n - g_{n-1}, sums over all cells and components,
 *           tau = (s.s)/(s.y) for odd n,  (s.y)/(y.y) for even n;
 *           if s.y <= 0 (or the quotient is not finite) tau = tau0; then clamp to [tau_min, tau_max]
 *   m_{n+1} = [ (1 - tau^2 |g_n|^2 / 4) m_n - tau g_n ] / (1 + tau^2 |g_n|^2 / 4)   per cell
 *           (|g| = |m x H| for unit m: the update is a rotation of m towards H, |m_{n+1}| = 1)
 *   dm_max = max over cells and components of |m_{n+1} - m_n|;  converged iff dm_max <= tol.
 * State carried between calls: n, m_prev, g_prev (caller-owned arrays of the size of m).
 * Outputs: *tau_used, *dm_max, *converged.  A call on a converged state is a no-op. */
typedef struct {
  long n;              /* iterations done */
  double tau0, tau_min, tau_max, tol;
  double tau, dm_max;  /* of the last iteration */
  int converged;
  double *m_prev, *g_prev;
} orc_bb_state;

int orc_bb_step(const orc_problem *p, double *m, orc_bb_state *st) {
  if (st->converged) return 0;
  const size_t n3 = (size_t)p->nx * p->ny * p->nz * 3;
  double *H = malloc(n3 * sizeof(double)), *g = malloc(n3 * sizeof(double));
  if (!H || !g) { free(H); free(g); return 2; }
  int rc = orc_heff(p, m, H);
  if (rc) { free(H); free(g); return rc; }
  for (size_t i = 0; i < n3; i += 3) {
    double mxh[3];
    cross3(m + i, H + i, mxh);
    cross3(m + i, mxh, g + i);
    if (p->Ms_cells && !(p->Ms_cells[i / 3] > 0.0)) g[i] = g[i + 1] = g[i + 2] = 0.0;   /* vacuum cell (O14) */
  }
  double tau = st->tau0;
  if (st->n > 0) {
    long double ss = 0.0L, sy = 0.0L, yy = 0.0L;
    for (size_t i = 0; i < n3; ++i) {
      const double s = m[i] - st->m_prev[i], y = g[i] - st->g_prev[i];
      ss += (long double)s * s; sy += (long double)s * y; yy += (long double)y * y;
    }
    const double q = (st->n & 1) ? (double)(ss / sy) : (double)(sy / yy);
    tau = (sy > 0.0L && isfinite(q)) ? q : st->tau0;
  }
  if (tau < st->tau_min) tau = st->tau_min;
  if (tau > st->tau_max) tau = st->tau_max;
  double dm = 0.0;
  for (size_t i = 0; i < n3; i += 3) {
    const double g2 = g[i] * g[i] + g[i + 1] * g[i + 1] + g[i + 2] * g[i + 2];
    const double a = 0.25 * tau * tau * g2;
    for (int c = 0; c < 3; ++c) {
      const double mn = ((1.0 - a) * m[i + c] - tau * g[i + c]) / (1.0 + a);
      const double d = fabs(mn - m[i + c]);
      if (d > dm) dm = d;
      st->m_prev[i + c] = m[i + c];
      st->g_prev[i + c] = g[i + c];
      m[i + c] = mn;
    }
  }
  st->n += 1;
  st->tau = tau;
  st->dm_max = dm;
  st->converged = dm <= st->tol ? 1 : 0;
  free(H); free(g);
  return 0;
}
