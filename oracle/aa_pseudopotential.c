/* CPU ORACLE -- TEST INFRASTRUCTURE ONLY (see arche_oracle.h).
 *
 * f2: norm-conserving pseudopotential from a finite-temperature Thomas-Fermi average atom
 * (Eq. 16-18), written from the paper in the order of its text:
 *   1. average-atom density n(r): one nucleus Z in a neutral Wigner-Seitz sphere of radius r_ws
 *      (4/3 pi rho r_ws^3 = 1), the same Thomas-Fermi relation Eq. 9 with the spherical potential
 *      V(r) = -Z/r + V_H[n](r) + V_xc(n(r)), mu from charge neutrality; solved self-consistently with the
 *      More et al. mixing the paper takes from the average-atom literature (Eq. 30-31, radial form);
 *   2. pseudo-density Eq. 16: exp(a + b r^2 + c r^4) inside r_cut, n(r) outside, with the three conditions of
 *      Eq. 17 (value, slope, charge inside r_cut);
 *   3. pseudopotential Eq. 18: the external potential for which the pseudo-density solves Eq. 9 in the sphere;
 *      it equals -Z/r for r >= r_cut (there the pseudo-density is the average-atom density);
 *   4. form factor V_s(k) = -Z/(pi k^2) + DV(k), DV(k) = int_0^r_cut (V_s(r) + Z/r) 4 pi r^2 sinc(2 pi k r) dr
 *      (the transform convention of PAPER.md:146), tabulated on a uniform k grid; DV(0) is the non-Coulomb k = 0
 *      constant alpha_s of Eq. 55.
 * Radial grid: uniform in x = sqrt(r) (r_i = (i h)^2, i = 0..n-1), which removes the r^(-3/2) singularity of the
 * Thomas-Fermi density at the nucleus from every integrand; integrals by the trapezoid rule in x with one
 * Richardson step (n must be odd).  Readings: DESIGN.md A22 (r_cut, energy definition, Hartree limits of Eq. 18).
 */
#include "arche_oracle.h"

#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

static const double PI = 3.14159265358979323846264338327950288;

/* Fermi-Dirac integrals over the range the average atom needs (eta up to ~1e6 at the nucleus).  oracle_fd's adaptive
 * quadrature is built for |eta| <~ 500 (its absolute tolerance drops below the rounding noise of the panels beyond
 * that, and it has no scale to stop on once I_j underflows), so outside that range the closed forms are used:
 * eta < -40: the first two terms of I_j = Gamma(j+1) sum_m (-1)^(m+1) e^(m eta)/m^(j+1) (third term < 1e-35 relative);
 * eta > 500: the Sommerfeld expansion
 *   I_j = eta^(j+1)/(j+1) [1 + sum_n 2 (1 - 2^(1-2n)) zeta(2n) (j+1) j (j-1) ... (j-2n+2) eta^(-2n)],  n = 1, 2, 3
 * (next term < 1e-17 relative at eta = 500; the exponentially small remainder is e^-500).  Exported for its pin. */
double oracle_fd_wide(int twice_j, double eta) {
  const double j = 0.5 * twice_j;
  if (eta < -40.0) {
    const double gam = twice_j == -1 ? sqrt(PI) : (twice_j == 1 ? 0.5 * sqrt(PI) : 0.75 * sqrt(PI)), x = exp(eta);
    return gam * x * (1.0 - x / pow(2.0, j + 1.0));
  }
  if (eta <= 500.0) return oracle_fd(twice_j, eta);
  const double e2 = 1.0 / (eta * eta);
  const double c1 = PI * PI / 6.0, c2 = 7.0 * PI * PI * PI * PI / 360.0, c3 = 31.0 * pow(PI, 6.0) / 15120.0;
  const double p1 = (j + 1.0) * j, p2 = p1 * (j - 1.0) * (j - 2.0), p3 = p2 * (j - 3.0) * (j - 4.0);
  return pow(eta, j + 1.0) / (j + 1.0) * (1.0 + e2 * (c1 * p1 + e2 * (c2 * p2 + e2 * c3 * p3)));
}
static double fd_safe(int twice_j, double eta) { return oracle_fd_wide(twice_j, eta); }
/* eta with I_{1/2}(eta) = y, any y > 0: bisection on oracle_fd_wide (same bounds as oracle_fd_half_inverse) */
double oracle_fd_half_inverse_wide(double y) {
  double g32 = 0.5 * sqrt(PI);
  double lo = log(y / g32), hi = pow(1.5 * y, 2.0 / 3.0) + 2.0;
  if (lo < -700.0) lo = -700.0;
  if (hi < lo + 2.0) hi = lo + 2.0;
  for (int it = 0; it < 200; ++it) {
    double mid = 0.5 * (lo + hi);
    if (mid == lo || mid == hi) break;
    if (oracle_fd_wide(1, mid) < y) lo = mid; else hi = mid;
  }
  return 0.5 * (lo + hi);
}

/* cumulative integral F_i = int_0^{x_i} g dx on the uniform x grid: Simpson on even nodes, Simpson + one 3/8-type
 * trapezoid-corrected step on odd nodes (fourth order everywhere except the first interval) */
static void cumint(int n, double h, const double *g, double *F) {
  F[0] = 0.0;
  if (n > 1) F[1] = h * (5.0 * g[0] + 8.0 * g[1] - g[2]) / 12.0; /* quadratic through the first three nodes */
  for (int i = 2; i < n; ++i) F[i] = F[i - 2] + h * (g[i - 2] + 4.0 * g[i - 1] + g[i]) / 3.0;
}

/* Hartree potential of a spherical density on the x grid: V_H(r) = (1/r) int_0^r 4 pi s^2 n ds + int_r^R 4 pi s n ds.
 * n0lim = lim r^(3/2) n(r) at r -> 0 (0 for a regular density). */
static void hartree(int n, double h, const double *r, const double *dens, double n0lim, double *VH, double *Qcum) {
  double *g1 = (double *)malloc(sizeof(double) * n), *g2 = (double *)malloc(sizeof(double) * n);
  double *I2 = (double *)malloc(sizeof(double) * n);
  for (int i = 0; i < n; ++i) {
    double x = i * h;
    g1[i] = i ? 8.0 * PI * x * x * x * x * x * dens[i] : 0.0;   /* 4 pi r^2 n dr, r = x^2, dr = 2 x dx */
    g2[i] = i ? 8.0 * PI * x * x * x * dens[i] : 8.0 * PI * n0lim; /* 4 pi r n dr */
  }
  cumint(n, h, g1, Qcum);
  cumint(n, h, g2, I2);
  for (int i = 0; i < n; ++i) VH[i] = (i ? Qcum[i] / r[i] : 0.0) + (I2[n - 1] - I2[i]);
  free(g1); free(g2); free(I2);
}

static double integrate(int n, double h, const double *g) {
  double *F = (double *)malloc(sizeof(double) * n);
  cumint(n, h, g, F);
  double v = F[n - 1];
  free(F);
  return v;
}

int oracle_aa_solve(double Z, double r_ws, double kT, int xc, int n, double *r, double *n_aa, double *mu_out,
                    int *iters_out) {
  if (n < 5 || !(n & 1) || !(Z > 0.0) || !(r_ws > 0.0) || !(kT > 0.0)) return -1;
  const double h = sqrt(r_ws) / (n - 1), cTF = sqrt(2.0) / (PI * PI) * pow(kT, 1.5);
  double *VH = (double *)malloc(sizeof(double) * n), *Q = (double *)malloc(sizeof(double) * n);
  double *na = (double *)malloc(sizeof(double) * n), *chi = (double *)malloc(sizeof(double) * n);
  double *V = (double *)malloc(sizeof(double) * n), *g = (double *)malloc(sizeof(double) * n);
  double *dVH = (double *)malloc(sizeof(double) * n), *dn = (double *)malloc(sizeof(double) * n);
  for (int i = 0; i < n; ++i) { r[i] = (i * h) * (i * h); n_aa[i] = 3.0 * Z / (4.0 * PI * r_ws * r_ws * r_ws); }
  n_aa[0] = 0.0;
  double mu = 0.0, n0lim = 0.0;
  int it, conv = 0;
  for (it = 1; it <= 2000; ++it) {
    hartree(n, h, r, n_aa, n0lim, VH, Q);
    for (int i = 1; i < n; ++i) {
      double e, v;
      oracle_xc(xc, n_aa[i], &e, &v);
      V[i] = -Z / r[i] + VH[i] + v;
    }
    /* mu from neutrality: N(mu) increasing; bracket and Illinois as in the 3D oracle */
    double lo = V[n - 1] - 60.0 * kT - 10.0 - 10.0 * Z * Z, hi = V[n - 1] + 60.0 * kT + 10.0 * Z;
    double flo = 0, fhi = 0;
    for (int pass = 0; pass < 2; ++pass) {
      double m = pass ? hi : lo;
#pragma omp parallel for schedule(dynamic, 16)
      for (int i = 1; i < n; ++i) { double x = i * h; g[i] = 8.0 * PI * x * x * x * x * x * cTF * fd_safe(1, (m - V[i]) / kT); }
      g[0] = 0.0;
      double f = integrate(n, h, g) - Z;
      if (pass) fhi = f; else flo = f;
    }
    if (!(flo < 0.0 && fhi > 0.0)) { conv = -2; break; }
    int side = 0;
    mu = lo;
    for (int k = 0; k < 200; ++k) {
      double x = (lo * fhi - hi * flo) / (fhi - flo);
      if (!(x > lo && x < hi)) x = 0.5 * (lo + hi);
#pragma omp parallel for schedule(dynamic, 16)
      for (int i = 1; i < n; ++i) { double xx = i * h; g[i] = 8.0 * PI * xx * xx * xx * xx * xx * cTF * fd_safe(1, (x - V[i]) / kT); }
      g[0] = 0.0;
      double fx = integrate(n, h, g) - Z;
      mu = x;
      if (fabs(fx) <= 1e-13 * Z || hi - lo <= 4e-16 * fmax(fabs(lo), fabs(hi))) break;
      if (fx > 0.0) { hi = x; fhi = fx; if (side == -1) flo *= 0.5; side = -1; }
      else { lo = x; flo = fx; if (side == +1) fhi *= 0.5; side = +1; }
    }
#pragma omp parallel for schedule(dynamic, 16)
    for (int i = 1; i < n; ++i) {
      double eta = (mu - V[i]) / kT;
      na[i] = cTF * fd_safe(1, eta);
      chi[i] = cTF * 0.5 * fd_safe(-1, eta) / kT;
    }
    na[0] = 0.0;
    /* More et al. (radial form): U = int dn dV_H, K = int dn^2/chi, w = U/(K+U) */
    double d2 = 0.0, a2 = 0.0;
    for (int i = 0; i < n; ++i) { dn[i] = n_aa[i] - na[i]; }
    hartree(n, h, r, dn, 0.0, dVH, Q);
    for (int i = 0; i < n; ++i) { double x = i * h; g[i] = i ? 8.0 * PI * x * x * x * x * x * dn[i] * dVH[i] : 0.0; }
    double U = integrate(n, h, g);
    for (int i = 0; i < n; ++i) { double x = i * h; g[i] = (i && chi[i] > 0.0) ? 8.0 * PI * x * x * x * x * x * dn[i] * dn[i] / chi[i] : 0.0; }
    double K = integrate(n, h, g);
    for (int i = 1; i < n; ++i) { double x = i * h, wgt = x * x * x * x * x; d2 += wgt * dn[i] * dn[i]; a2 += wgt * na[i] * na[i]; }
    double w = (it <= 3) ? 0.5 : ((K + U > 0.0) ? U / (K + U) : 0.0);
    for (int i = 0; i < n; ++i) n_aa[i] = na[i] + w * (n_aa[i] - na[i]);
    /* limit of r^(3/2) n at the nucleus: degenerate Thomas-Fermi, n -> (2 Z/r)^(3/2)/(3 pi^2) */
    n0lim = pow(2.0 * Z, 1.5) / (3.0 * PI * PI);
    if (getenv("ORACLE_AA_DEBUG")) fprintf(stderr, "aa it %d mu %.10f w %.6f res %.3e U %.3e K %.3e\n", it, mu, w, sqrt(d2 / a2), U, K);
    if (sqrt(d2 / a2) < 1e-12) { conv = 1; break; }
  }
  /* return the ACTIVE density of the last iteration (it satisfies Eq. 9 with the potential of the mixed input) */
  for (int i = 0; i < n; ++i) n_aa[i] = na[i];
  *mu_out = mu;
  if (iters_out) *iters_out = it;
  free(VH); free(Q); free(na); free(chi); free(V); free(g); free(dVH); free(dn);
  return conv == 1 ? 0 : -3;
}

/* Eq. 16-17: a, b, c of exp(a + b r^2 + c r^4) from the value and slope of n at r_cut = r[ic] and the charge inside */
int oracle_aa_pseudize(int n, const double *r, const double *n_aa, int ic, double *n_ps, double abc[3]) {
  if (ic < 4 || ic >= n - 2 || !(n & 1)) return -1;
  const double h = sqrt(r[n - 1]) / (n - 1), rc = r[ic];
  /* slope dn/dr at r_cut from the x grid: dn/dx by the 4th-order central difference, dr = 2 x dx */
  double xc_ = ic * h;
  double dndx = (n_aa[ic - 2] - 8.0 * n_aa[ic - 1] + 8.0 * n_aa[ic + 1] - n_aa[ic + 2]) / (12.0 * h);
  double nc = n_aa[ic], slope = dndx / (2.0 * xc_);
  /* charge inside r_cut of the average atom */
  double *g = (double *)malloc(sizeof(double) * n);
  for (int i = 0; i <= ic; ++i) { double x = i * h; g[i] = i ? 8.0 * PI * x * x * x * x * x * n_aa[i] : 0.0; }
  /* integrate on [0, x_c]: needs an odd number of nodes; if ic is odd, add the last panel by the 3-point rule */
  double Qaa;
  {
    double *F = (double *)malloc(sizeof(double) * (ic + 1));
    cumint(ic + 1, h, g, F);
    Qaa = F[ic];
    free(F);
  }
  /* for given c: b from the slope, a from the value; Q(c) decreasing in c?  solve Q(c) = Qaa by bracketing + bisection */
  double L = log(nc), s = slope / nc; /* d ln n / dr */
  double clo = -50.0 / (rc * rc * rc * rc), chi_ = 50.0 / (rc * rc * rc * rc), c = 0.0, a = 0.0, b = 0.0;
  double flo = 0.0, fhi = 0.0;
  for (int pass = 0; pass < 202; ++pass) {
    double cc = pass == 0 ? clo : (pass == 1 ? chi_ : 0.5 * (clo + chi_));
    double bb = (s - 4.0 * cc * rc * rc * rc) / (2.0 * rc), aa = L - bb * rc * rc - cc * rc * rc * rc * rc;
    for (int i = 0; i <= ic; ++i) {
      double x = i * h, rr = x * x;
      g[i] = 8.0 * PI * x * x * x * x * x * exp(aa + bb * rr * rr + cc * rr * rr * rr * rr);
    }
    double *F = (double *)malloc(sizeof(double) * (ic + 1));
    cumint(ic + 1, h, g, F);
    double f = F[ic] - Qaa;
    free(F);
    if (pass == 0) { flo = f; continue; }
    if (pass == 1) { fhi = f; if (!(flo * fhi < 0.0)) { free(g); return -2; } continue; }
    c = cc; a = aa; b = bb;
    if (fabs(f) <= 1e-14 * Qaa || chi_ - clo <= 1e-16 * fabs(chi_)) break;
    if ((f > 0.0) == (fhi > 0.0)) { chi_ = cc; fhi = f; } else { clo = cc; flo = f; }
  }
  for (int i = 0; i < n; ++i) n_ps[i] = i <= ic ? exp(a + b * r[i] * r[i] + c * r[i] * r[i] * r[i] * r[i]) : n_aa[i];
  abc[0] = a; abc[1] = b; abc[2] = c;
  free(g);
  return 0;
}

/* Eq. 18: the external potential for which `dens` solves Eq. 9 in the sphere with chemical potential mu:
 * V_ext(r) = mu - kT I_{1/2}^{-1}(dens/cTF) - V_H[dens](r) - V_xc(dens).  n0lim as in hartree(). */
int oracle_aa_invert(double kT, int xc, int n, const double *r, const double *dens, double n0lim, double mu, double *V_ext) {
  if (n < 5 || !(n & 1)) return -1;
  const double h = sqrt(r[n - 1]) / (n - 1), cTF = sqrt(2.0) / (PI * PI) * pow(kT, 1.5);
  double *VH = (double *)malloc(sizeof(double) * n), *Q = (double *)malloc(sizeof(double) * n);
  hartree(n, h, r, dens, n0lim, VH, Q);
#pragma omp parallel for schedule(dynamic, 16)
  for (int i = 1; i < n; ++i) {
    double e, v;
    oracle_xc(xc, dens[i], &e, &v);
    V_ext[i] = mu - kT * oracle_fd_half_inverse_wide(dens[i] / cTF) - VH[i] - v;
  }
  V_ext[0] = V_ext[1];
  free(VH); free(Q);
  return 0;
}

/* DV(k) = int_0^{r[ic]} f(r) 4 pi r^2 sin(2 pi k r)/(2 pi k r) dr on the x grid (PAPER.md:146 convention) */
void oracle_radial_ft(int n, const double *r, const double *f, int ic, int nk, const double *k, double *out) {
  const double h = sqrt(r[n - 1]) / (n - 1);
#pragma omp parallel for schedule(static)
  for (int m = 0; m < nk; ++m) {
    double *g = (double *)malloc(sizeof(double) * (ic + 1)), *F = (double *)malloc(sizeof(double) * (ic + 1));
    for (int i = 0; i <= ic; ++i) {
      double x = i * h, q = 2.0 * PI * k[m] * r[i];
      double sinc = q > 1e-6 ? sin(q) / q : 1.0 - q * q / 6.0;
      g[i] = 8.0 * PI * x * x * x * x * x * f[i] * sinc;
    }
    cumint(ic + 1, h, g, F);
    out[m] = F[ic];
    free(g); free(F);
  }
}

/* Average-atom internal energy of a density in the sphere with external potential -Z/r (Coulomb) or a given V_ext:
 * E = K_e + int n V_ext + (1/2) int n V_H + E_xc, K_e = int kT cTF I_{3/2}(eta) with eta the Thomas-Fermi variable of
 * the density, eta = I_{1/2}^{-1}(n/cTF) (Eq. 38).  out[4] = {K_e, E_ext, E_H, E_xc}. */
int oracle_aa_energy(double kT, int xc, int n, const double *r, const double *dens, double n0lim, const double *V_ext,
                     double Zc, double out[4]) {
  if (n < 5 || !(n & 1)) return -1;
  const double h = sqrt(r[n - 1]) / (n - 1), cTF = sqrt(2.0) / (PI * PI) * pow(kT, 1.5);
  double *VH = (double *)malloc(sizeof(double) * n), *Q = (double *)malloc(sizeof(double) * n);
  double *g = (double *)malloc(sizeof(double) * n), *ke = (double *)malloc(sizeof(double) * n);
  hartree(n, h, r, dens, n0lim, VH, Q);
#pragma omp parallel for schedule(dynamic, 16)
  for (int i = 1; i < n; ++i) ke[i] = kT * cTF * oracle_fd_wide(3, oracle_fd_half_inverse_wide(dens[i] / cTF));
  /* K_e: near the nucleus ke -> (3/10)(3 pi^2)^(2/3) n^(5/3) ~ r^(-5/2) (degenerate limit): 8 pi x^5 ke is finite at 0 */
  double lim_ke = 0.3 * pow(3.0 * PI * PI, 2.0 / 3.0) * pow(n0lim, 5.0 / 3.0);
  for (int i = 0; i < n; ++i) { double x = i * h; g[i] = i ? 8.0 * PI * x * x * x * x * x * ke[i] : 8.0 * PI * lim_ke; }
  out[0] = integrate(n, h, g);
  for (int i = 0; i < n; ++i) {
    double x = i * h;
    if (V_ext) g[i] = i ? 8.0 * PI * x * x * x * x * x * dens[i] * V_ext[i] : 0.0;
    else g[i] = i ? -Zc * 8.0 * PI * x * x * x * dens[i] : -Zc * 8.0 * PI * n0lim;   /* n (-Z/r) 4 pi r^2 dr = -Z 8 pi x^3 n dx */
  }
  out[1] = integrate(n, h, g);
  for (int i = 0; i < n; ++i) { double x = i * h; g[i] = i ? 4.0 * PI * x * x * x * x * x * dens[i] * VH[i] : 0.0; }
  out[2] = integrate(n, h, g);
  for (int i = 0; i < n; ++i) {
    double x = i * h, e = 0.0, v = 0.0;
    if (i) oracle_xc(xc, dens[i], &e, &v);
    g[i] = i ? 8.0 * PI * x * x * x * x * x * dens[i] * e : 0.0;
  }
  out[3] = integrate(n, h, g);
  free(VH); free(Q); free(g); free(ke);
  return 0;
}
