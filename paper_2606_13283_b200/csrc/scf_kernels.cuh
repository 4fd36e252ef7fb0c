// scf_kernels.cuh -- SCF-iteration kernels and the pointwise functors of steps S1..S7:
// potential assembly in G-space, V_i epilogue with XC, device-side secant/Newton-in-bracket for mu (Eq. 19), density
// and local reductions, G-space reductions, mixing.  The functors run in three hosts: fused into the FFT passes
// (fft_fast.cuh, fft.cuh), in the streaming kernels below (large grids), and in the persistent kernel
// (scf_persistent.cuh).
#pragma once
#include "common.cuh"
#include "fd.cuh"
#include "fft.cuh"
#include <cooperative_groups.h>

namespace arche {

// All scalars of one solve live in this device struct; the host reads it back once per SCF iteration.
struct DevScalars {
  // S2 epilogue
  double vmin, vmax, vsum;
  // S3 state
  double mu, mu_lo, mu_hi, N_last, dNdmu, n0sum;
  int mu_done, mu_evals, mu_have_prev, pad0;
  // S4
  double K, dn2, na2, F0, Ke, Exc;
  // S5
  double U, EH, Eie;
  // S6/S7
  double w, F_total, F_prev, dn_rel;
  int iter, converged, mu_evals_total, flip_seen;   // flip_seen: reading A13, a PZ81 branch flip was detected in this solve
  int more_on, pad1;                                // reading A11b: More's w has been switched on in this solve
  double mu_iter_prev, tolF_eff, toldn_eff;         // mu_a of the previous iteration; the tolerances the stop rule applied
  // per-MD-step
  double U_pp, U_pm_sum, U_pm_fix, U_ii, init_sum, init_scale, K_i;
  // lazy free energy (ScfConst::lazy_F): skip_F = the running iteration leaves out the terms only F needs (I_{3/2}, eps_xc,
  // E_ie); F_valid = F_total is the free energy of the previous iteration
  int skip_F, F_valid, F_evals, pad2;   // F_evals: iterations of this solve that evaluated the free energy
};

struct ScfConst {
  double kT, cTF, Ne, vol, dV, eta0, E_ie0;
  int xc, mix_mode, mix_warmup;
  int lazy_F;   // > 0: solves under the stop rule evaluate the free energy only from the iteration at which the density
                // criterion is predicted to be met within two iterations, and in iteration lazy_F (= scf_max_iter), so that
                // a solve never ends without it.  The paper's own stop rule needs no F; BASELINE's |dF| criterion
                // needs F_k and F_{k-1} of the last two iterations only.  0: every iteration (parity replays, xc = 1)
  double mix_w_fixed, tol_F, tol_dn;
  double inv_vol, inv_qF;   // reciprocals for the single-thread scalar updates (fp64 divisions cost ~300 cycles each there)
  double q_F, q_dn;   // reading A13: free-energy quantum of one PZ81 branch flip; chi(n*) x V_c jump x sqrt(dV)
  double mix_mu_tol;  // reading A11b: More's w only once |mu_k - mu_{k-1}| <= mix_mu_tol kT (latched); <= 0: off
  double chi_floor;   // reading A11c: lower bound of dn_a/dmu in K (Eq. 31), absolute; 0: Eq. 31 as printed
};

// Perdew-Zunger 1981 LDA (unpolarised), Hartree units; restated from the publication (reading D5).
// One reciprocal cube root gives r_s and n^(1/3) (no division), one reciprocal serves eps_c and V_c on the r_s >= 1
// branch; the branch is decided on r_s in fp64 exactly as in the oracle (reading A13).
// xc = 1: the constants as printed (C = 0.0020, D = -0.0116: eps_c and V_c jump by ~3e-5 Ha at r_s = 1);
// xc = 2: C and D at full precision from the two matching conditions Perdew and Zunger imposed at r_s = 1 (eps_c and
//         d eps_c/d r_s continuous) with the other five printed constants -- they round to the printed values; eps_c and
//         V_c are then continuous and the SCF has a fixed point on every grid (reading A13b).
namespace pz81 {
constexpr double g = -0.1423, b1 = 1.0529, b2 = 0.3334, A = 0.0311, B = -0.048;
constexpr double den1 = 1.0 + b1 + b2, ec1 = g / den1, dec1 = -g * (0.5 * b1 + b2) / (den1 * den1);
constexpr double D_mod = ec1 - B, C_mod = dec1 - A - D_mod;   // 0.0020191519..., -0.0116320663...
}  // namespace pz81
// 1/x for normal x: MUFU.RCP64H seed (20 bits) + two Newton steps (4 DFMA), branch-free.  The compiler's fp64 division
// and __drcp_rn carry a slow-path branch and ~2x the instructions; the result here is within 1 ulp.
__device__ __forceinline__ double rcp_fast(double x) {
  double r;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
  double e = fma(-x, r, 1.0);
  r = fma(r, e, r);
  e = fma(-x, r, 1.0);
  return fma(r, e, r);
}
// u = n^(-1/6) for n >= 1e-250: every power PZ81 needs is a product of u (r_s = c u^2, sqrt r_s = sqrt(c) u,
// n^(1/3) = n u^4), so one Newton iteration chain replaces a cube root and a square root.  The argument is first
// brought into [1, 64) by an exact power of two taken from its exponent field (n = ns 2^(6k), u = u(ns) 2^(-k)): the
// densities of a degenerate plasma span 1e-100 ... 10 (empty cores at T = 1 eV) and an fp32 seed of n itself would
// underflow.  fp32 seed exp2(-log2(ns)/6) (two MUFU), two steps of u <- u + u (1 - ns u^6)/6 (quadratic:
// 1e-6 -> 4e-12 -> round-off).
__device__ __forceinline__ double inv_sixth_root(double n) {
  const int e = (__double2hiint(n) >> 20) - 1023;      // n > 0, normal: sign bit clear
  const int k = (e >= 0 ? e : e - 5) / 6;              // floor(e / 6)
  const double ns = n * __hiloint2double((1023 - 6 * k) << 20, 0);
  double u = (double)exp2f(__log2f((float)ns) * (-1.0f / 6.0f));
#pragma unroll
  for (int it = 0; it < 2; ++it) {
    const double u2 = u * u, u6 = u2 * u2 * u2;
    u = fma(u * (1.0 / 6.0), fma(-ns, u6, 1.0), u);
  }
  return u * __hiloint2double((1023 - k) << 20, 0);
}
__device__ __forceinline__ void xc_pz81(double n, double &eps, double &v, int xc = 1) {
  // below 1e-250 the potential -(3n/pi)^(1/3) is < 1e-83 Ha and the energy density n eps_xc < 1e-333: taken as zero
  if (!(n > 1.0e-250)) { eps = 0.0; v = 0.0; return; }
  const double cx = 0.73855876638202240588;   // (3/4) (3/pi)^(1/3)
  const double c0 = 0.62035049089940001667;   // (3/(4 pi))^(1/3): r_s = c0 n^(-1/3)
  const double sc0 = 0.78762331789974325053;  // sqrt(c0)
  const double u = inv_sixth_root(n), u2 = u * u;
  const double ex = -cx * (n * (u2 * u2));
  const double rs = c0 * u2;
  double ec, vc;
  if (rs >= 1.0) {
    const double a1 = pz81::b1 * sc0, a2 = pz81::b2 * c0;     // beta1 sqrt(r_s) = a1 u, beta2 r_s = a2 u^2
    const double inv = rcp_fast(fma(a2, u2, fma(a1, u, 1.0)));
    ec = pz81::g * inv;
    vc = ec * fma((4.0 / 3.0) * a2, u2, fma((7.0 / 6.0) * a1, u, 1.0)) * inv;
  } else {
    const double A = pz81::A, B = pz81::B, C = xc == 2 ? pz81::C_mod : 0.0020, D = xc == 2 ? pz81::D_mod : -0.0116;
    const double l = log(rs);
    ec = A * l + B + C * rs * l + D * rs;
    vc = A * l + (B - A / 3.0) + (2.0 / 3.0) * C * rs * l + (2.0 * D - C) / 3.0 * rs;
  }
  eps = ex + ec;
  v = (4.0 / 3.0) * ex + vc;
}

// Half-spectrum conventions (fft.cuh): G-space arrays are [nz][ny][P], ix = 0..nx/2 stored.  A sum over the full
// reciprocal grid is sum_half wt(ix) (...), wt = 1 on the self-mirrored columns ix = 0 and (even nx) ix = nx/2, else 2.
struct HalfGeom {
  int nx, nxh;  // nxh = nx/2 + 1
  __device__ __forceinline__ double wt(int ix) const { return (ix == 0 || 2 * ix == nx) ? 1.0 : 2.0; }
};

// ---- S1: Vhat(k) = nhat_i(k)/(pi k^2) + Vhat_ie(k), 0 at k = 0 (Eq. 12, 14).  When a mixing step is pending the
// new input density nhat_i <- nhat_a + w (nhat_i - nhat_a) (S6) is formed here and written back.
struct LoadPotentialG {
  static constexpr bool kWriteBack = true;
  double2 *nh_i;
  const double2 *nh_a, *vh_ie;
  const double *kx2, *ky2, *kz2;
  const DevScalars *sc;
  int nxh, mix;
  double w;
  __device__ __forceinline__ void begin() { w = mix ? sc->w : 1.0; }
  __device__ __forceinline__ void prefetch(long long idx) const {
    prefetch_l2(nh_i + idx); prefetch_l2(vh_ie + idx);
    if (mix) prefetch_l2(nh_a + idx);
  }
  __device__ __forceinline__ void operator()(long long idx, int ix, int iy, int iz, double &re, double &im) {
    if (ix >= nxh) { re = 0.0; im = 0.0; return; }
    double2 a = nh_i[idx];
    if (mix) {
      const double2 na = nh_a[idx];
      a = make_double2(fma(w, a.x - na.x, na.x), fma(w, a.y - na.y, na.y));
      nh_i[idx] = a;
    }
    const double k2 = kx2[ix] + ky2[iy] + kz2[iz];
    if (k2 == 0.0) { re = 0.0; im = 0.0; return; }
    const double inv = __drcp_rn(ARCHE_PI * k2);
    const double2 b = vh_ie[idx];
    re = fma(a.x, inv, b.x); im = fma(a.y, inv, b.y);
  }
  // the same without the in-place store: wb receives the mixed nhat_i, stored afterwards by store_wb
  __device__ __forceinline__ void load_wb(long long idx, int ix, int iy, int iz, double &re, double &im, double2 &wb) {
    re = 0.0; im = 0.0; wb = make_double2(0.0, 0.0);
    if (ix >= nxh) return;
    double2 a = nh_i[idx];
    if (mix) {
      const double2 na = nh_a[idx];
      a = make_double2(fma(w, a.x - na.x, na.x), fma(w, a.y - na.y, na.y));
    }
    wb = a;
    const double k2 = kx2[ix] + ky2[iy] + kz2[iz];
    if (k2 == 0.0) return;
    const double inv = __drcp_rn(ARCHE_PI * k2);
    const double2 b = vh_ie[idx];
    re = fma(a.x, inv, b.x); im = fma(a.y, inv, b.y);
  }
  __device__ __forceinline__ void store_wb(long long idx, int ix, double2 wb) { if (mix && ix < nxh) nh_i[idx] = wb; }
  __device__ __forceinline__ void finish(double *) {}
};

// ---- S2: V_i = IFFT/|Omega| + V_xc(n_i); min/max/sum of V_i; the last block opens the mu bracket.  A pending
// mixing step forms the real-space n_i here (S6).  When a previous mu exists the first Newton evaluation
// sum I_{1/2}((mu_prev - V_i)/kT) is taken in the same pass (S3).
struct StoreVi {
  double *V_i, *n_i;
  const double *n_a;
  DevScalars *sc;
  double *partials;
  unsigned int *counter;
  const double *fdtab;
  double inv_vol, kT_eta0, inv_kT;
  int xc, mix;
  double w, mu0, acc_min, acc_max, acc_sum, acc_n;
  int have_mu;
  __device__ __forceinline__ void set_table(const double *t) { fdtab = t; }
  __device__ __forceinline__ void begin() {
    w = mix ? sc->w : 1.0;
    have_mu = sc->mu_have_prev; mu0 = sc->mu;
    acc_min = 1.0e308; acc_max = -1.0e308; acc_sum = 0.0; acc_n = 0.0;
  }
  __device__ __forceinline__ void prefetch(long long idx) const {
    prefetch_l2(n_i + idx);
    if (mix) prefetch_l2(n_a + idx);
  }
  __device__ __forceinline__ void store_real(long long idx, int, int, int, double re) {
    double v = re * inv_vol;
    double ni = n_i[idx];
    if (mix) { const double na = n_a[idx]; ni = fma(w, ni - na, na); n_i[idx] = ni; }
    if (xc) { double e, vx; xc_pz81(ni, e, vx, xc); v += vx; }
    V_i[idx] = v;
    acc_min = fmin(acc_min, v); acc_max = fmax(acc_max, v); acc_sum += v;
    if (have_mu) { double a, b, c; fd_eval<2>(fdtab, (mu0 - v) * inv_kT, a, b, c); acc_n += b; }
  }
  // two elements at once (the two lines of an x-pass pair): interleaves the two Fermi-Dirac evaluations.  Split into
  // fetch (the global loads) and compute so that the streaming kernel can issue the next pair's loads before it works
  // on the current pair.
  struct Pre { double ni0, ni1, na0, na1; };
  __device__ __forceinline__ void fetch(long long ia, long long ib, Pre &p) const {
    p.ni0 = n_i[ia]; p.ni1 = n_i[ib];
    if (mix) { p.na0 = n_a[ia]; p.na1 = n_a[ib]; }
  }
  __device__ __forceinline__ void compute(long long ia, long long ib, const Pre &p, double ra, double rb) {
    double v[2] = {ra * inv_vol, rb * inv_vol};
    double ni[2] = {p.ni0, p.ni1};
    if (mix) {
      ni[0] = fma(w, ni[0] - p.na0, p.na0); ni[1] = fma(w, ni[1] - p.na1, p.na1);
      n_i[ia] = ni[0]; n_i[ib] = ni[1];
    }
    if (xc) {
      double e, vx;
      xc_pz81(ni[0], e, vx, xc); v[0] += vx;
      xc_pz81(ni[1], e, vx, xc); v[1] += vx;
    }
    V_i[ia] = v[0]; V_i[ib] = v[1];
    acc_min = fmin(acc_min, fmin(v[0], v[1])); acc_max = fmax(acc_max, fmax(v[0], v[1])); acc_sum += v[0]; acc_sum += v[1];
    if (have_mu) {
      double eta[2] = {(mu0 - v[0]) * inv_kT, (mu0 - v[1]) * inv_kT}, a[2], b[2], c[2];
      fd_eval_multi<2, 2>(fdtab, eta, a, b, c);
      acc_n += b[0]; acc_n += b[1];
    }
  }
  __device__ __forceinline__ void store_real2(long long ia, long long ib, double ra, double rb) {
    Pre p; fetch(ia, ib, p); compute(ia, ib, p, ra, rb);
  }
  __device__ __forceinline__ void finish(double *smem) {
    double v[4] = {acc_min, acc_max, acc_sum, acc_n};
    const int op[4] = {1, 2, 0, 0};
    if (grid_reduce<4>(v, op, partials, counter, smem) && threadIdx.x == 0) apply(smem + 4 * 32, kT_eta0, sc);
  }
  // grid totals {min, max, sum of V_i, sum I_{1/2}} -> scalars and the mu bracket
  static __device__ __forceinline__ void apply(const double *t, double kT_eta0, DevScalars *sc) {
    sc->vmin = t[0]; sc->vmax = t[1]; sc->vsum = t[2]; sc->n0sum = t[3];
    sc->mu_done = 0;   // a new potential: the mu iteration of this SCF iteration has not run yet
    // bracket of the root of Eq. 19: N(mu) is increasing and eta0 solves the flat-potential problem
    const double lo = t[0] + kT_eta0, hi = t[1] + kT_eta0;
    const double pad = 1e-12 * (fabs(lo) + fabs(hi) + fabs(kT_eta0));
    sc->mu_lo = lo - pad; sc->mu_hi = hi + pad;
  }
  // persistent form: block partial sums only (the totals are taken by every block after the next grid barrier)
  __device__ __forceinline__ void partial(double *smem, double *out /*[gridDim.x][4]*/) {
    double v[4] = {acc_min, acc_max, acc_sum, acc_n};
    const int op[4] = {1, 2, 0, 0};
    block_partials<4>(v, op, smem, out);
  }
};

// ---- S3: mu from charge neutrality (Eq. 19), persistent cooperative kernel.  Newton-type iteration kept inside
// the bracket (reading D1): the first evaluation comes from the S2 pass when a previous mu exists (slope = dN/dmu of
// the previous density pass), later slopes are secants; one grid-wide barrier per evaluation.  Every block re-sums
// all block partials in the same fixed order, so all blocks take the same step.  On small grids the V_i values of a
// thread stay in registers across the passes.
constexpr int kMuCache = 8;
// sum of I_{1/2} (and I_{-1/2} when SLOPE) over four potentials at once
template <bool SLOPE>
__device__ __forceinline__ void mu_accumulate4(const double *tab, const double (&v)[4], const bool (&ok)[4], double mu,
                                               double inv_kT, double &s1, double &s0) {
  double eta[4], im12[4] = {0.0, 0.0, 0.0, 0.0}, i12[4], d[4];
#pragma unroll
  for (int q = 0; q < 4; ++q) eta[q] = ok[q] ? (mu - v[q]) * inv_kT : 1.0;
  fd_eval_multi<SLOPE ? 3 : 2, 4>(tab, eta, im12, i12, d);
#pragma unroll
  for (int q = 0; q < 4; ++q) if (ok[q]) { s1 += i12[q]; s0 += im12[q]; }
}

constexpr size_t kFdTabBytes = sizeof(double) * kFdTabDoubles;
// s_tab: the Fermi-Dirac table in shared memory (already loaded and synchronised); s_red: [2*32+2]; s_bc: [2];
// partials: [2][gridDim.x][2], not shared with any other reduction that may run concurrently; sc may be the global
// scalar block (block 0 writes the result) or a per-block shared copy (sc_is_block_local: every block writes its own)
__device__ __forceinline__ double mu_solve_dev(cooperative_groups::grid_group &grid, const double *__restrict__ V_i,
                                             long long ng, const ScfConst &C, DevScalars *sc, const double *s_tab,
                                             double *s_red, double *s_bc, double *partials, int max_pass,
                                             bool sc_is_block_local = false) {
  const double inv_kT = 1.0 / C.kT, kT_eta0 = C.kT * C.eta0, scaleN = C.cTF * C.dV;
  const long long nthreads = (long long)gridDim.x * blockDim.x, tid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const bool cached = ng <= nthreads * kMuCache;
  double vc[kMuCache];
  if (cached) {
#pragma unroll
    for (int q = 0; q < kMuCache; ++q) { long long g = tid + q * nthreads; vc[q] = g < ng ? V_i[g] : 0.0; }
  }
  __syncthreads();
  double lo = sc->mu_lo, hi = sc->mu_hi;
  const int have_prev = sc->mu_have_prev;
  double mu, f = 0.0, slope = 0.0;
  bool have_f = false, done = false, slope_fresh = false;   // slope_fresh: exact or secant (not the previous iteration's)
  int evals = 0;
  if (hi - lo <= 4e-16 * fmax(fabs(lo), fabs(hi))) { mu = 0.5 * (lo + hi); done = true; }  // flat potential
  else if (have_prev) { mu = sc->mu; f = scaleN * sc->n0sum - C.Ne; slope = sc->dNdmu; have_f = slope > 0.0; evals = have_f; }
  else mu = sc->vsum / (double)ng + kT_eta0;
  if (!done && !have_f && !(mu > lo && mu < hi)) mu = 0.5 * (lo + hi);
  double mu_prev = mu, f_prev = 0.0;
  bool have_prev_pt = false;
  for (int pass = 0; pass < max_pass && !done; ++pass) {
    if (!have_f) {
      const bool want_slope = !(slope > 0.0);
      double s1 = 0.0, s0 = 0.0;
      if (cached) {
#pragma unroll
        for (int h = 0; h < kMuCache; h += 4) {
          bool ok[4]; double vv[4];
#pragma unroll
          for (int q = 0; q < 4; ++q) { ok[q] = tid + (h + q) * nthreads < ng; vv[q] = vc[h + q]; }
          if (!ok[0]) break;
          if (want_slope) mu_accumulate4<true>(s_tab, vv, ok, mu, inv_kT, s1, s0);
          else mu_accumulate4<false>(s_tab, vv, ok, mu, inv_kT, s1, s0);
        }
      } else if (!(ng & 1)) {
        // streaming pass, lean form (ncu, round 2: this loop issued 74 instructions per point, 55 of them integer/select
        // bookkeeping on the ALU pipe): 32-bit indices, 16-byte loads of two potentials, no per-element predicates in
        // the body, the Fermi-Dirac argument from one FMA, the next group's loads in flight during the evaluation
        const double sA = inv_kT * FD_INV_W, sB = (mu * inv_kT - FD_ETA_A) * FD_INV_W;   // s = sB - v sA
        const double2 *V2 = reinterpret_cast<const double2 *>(V_i);
        const int n2 = (int)(ng >> 1), nth = (int)nthreads;
        int i = (int)tid;
        const double2 zero2 = make_double2(0.0, 0.0);
        double2 a = i < n2 ? V2[i] : zero2, b = i + nth < n2 ? V2[i + nth] : zero2;
        for (; i < n2; i += 2 * nth) {
          const int in = i + 2 * nth;
          const double2 an = in < n2 ? V2[in] : zero2, bn = in + nth < n2 ? V2[in + nth] : zero2;
          if (i + nth < n2) {
            const double sg[4] = {fma(-a.x, sA, sB), fma(-a.y, sA, sB), fma(-b.x, sA, sB), fma(-b.y, sA, sB)};
            double im12[4], i12[4], d[4];
            fd_eval_multi_s<2, 4>(s_tab, sg, im12, i12, d);
            s1 += (i12[0] + i12[1]) + (i12[2] + i12[3]);
            if (want_slope) {   // rare (first pass without a previous slope): a second sweep over the same arguments
              fd_eval_multi_s<1, 4>(s_tab, sg, im12, i12, d);
              s0 += (im12[0] + im12[1]) + (im12[2] + im12[3]);
            }
          } else {
            const double sg[2] = {fma(-a.x, sA, sB), fma(-a.y, sA, sB)};
            double im12[2] = {0.0, 0.0}, i12[2], d[2];
            if (want_slope) fd_eval_multi_s<3, 2>(s_tab, sg, im12, i12, d);
            else fd_eval_multi_s<2, 2>(s_tab, sg, im12, i12, d);
            s1 += i12[0] + i12[1]; s0 += im12[0] + im12[1];
          }
          a = an; b = bn;
        }
      } else {
        // odd point count (all three axes powers of 3): element-wise form
        double va[4], vb[4];
#pragma unroll
        for (int q = 0; q < 4; ++q) {
          const long long ga = tid + q * nthreads, gb = ga + 4 * nthreads;
          va[q] = ga < ng ? V_i[ga] : 0.0; vb[q] = gb < ng ? V_i[gb] : 0.0;
        }
        for (long long g0 = tid; g0 < ng; g0 += 8 * nthreads) {
          double vv[4]; bool ok[4];
#pragma unroll
          for (int q = 0; q < 4; ++q) {
            const long long g = g0 + q * nthreads, gn = g + 8 * nthreads;
            ok[q] = g < ng; vv[q] = va[q]; va[q] = gn < ng ? V_i[gn] : 0.0;
          }
          if (want_slope) mu_accumulate4<true>(s_tab, vv, ok, mu, inv_kT, s1, s0);
          else mu_accumulate4<false>(s_tab, vv, ok, mu, inv_kT, s1, s0);
          if (g0 + 4 * nthreads >= ng) break;
#pragma unroll
          for (int q = 0; q < 4; ++q) {
            const long long g = g0 + (4 + q) * nthreads, gn = g + 8 * nthreads;
            ok[q] = g < ng; vv[q] = vb[q]; vb[q] = gn < ng ? V_i[gn] : 0.0;
          }
          if (want_slope) mu_accumulate4<true>(s_tab, vv, ok, mu, inv_kT, s1, s0);
          else mu_accumulate4<false>(s_tab, vv, ok, mu, inv_kT, s1, s0);
        }
      }
      double v[2] = {s1, s0};
      const int op[2] = {0, 0};
      block_reduce<2>(v, op, s_red);
      double *buf = partials + (size_t)(pass & 1) * 2 * gridDim.x;
      if (threadIdx.x == 0) { buf[2 * blockIdx.x] = v[0]; buf[2 * blockIdx.x + 1] = v[1]; }
      grid.sync();
      double a[2] = {0.0, 0.0};
      for (unsigned int b = threadIdx.x; b < gridDim.x; b += blockDim.x) { a[0] += __ldcg(&buf[2 * b]); a[1] += __ldcg(&buf[2 * b + 1]); }
      block_reduce<2>(a, op, s_red);
      if (threadIdx.x == 0) { s_bc[0] = a[0]; s_bc[1] = a[1]; }
      __syncthreads();
      f = scaleN * s_bc[0] - C.Ne;
      if (want_slope) { slope = scaleN * 0.5 * s_bc[1] * inv_kT; slope_fresh = true; }           // dN/dmu (I_j' = j I_{j-1})
      else if (have_prev_pt && mu != mu_prev) { const double sct = (f - f_prev) / (mu - mu_prev); if (sct > 0.0) { slope = sct; slope_fresh = true; } }
      __syncthreads();
      ++evals;
    }
    have_f = false;
    if (fabs(f) <= 1e-14 * C.Ne || pass == max_pass - 1) { done = true; break; }
    if (f > 0.0) hi = fmin(hi, mu); else lo = fmax(lo, mu);
    double mu_new = mu - f / slope;
    if (!(mu_new > lo && mu_new < hi)) mu_new = 0.5 * (lo + hi);
    if (fabs(mu_new - mu) <= 2e-16 * fmax(fabs(mu), C.kT)) { done = true; break; }
    // With an exact or secant slope the residual after the step is ~ f (f''/2f') max(|step|, |previous step|)
    // <= |f| max(step)/kT (I_{-1/2}'/I_{-1/2} <= 1/2 per kT): when that is below the tolerance the step is taken
    // without another pass over the grid (the density pass that follows evaluates at the accepted mu).
    if (slope_fresh) {
      const double st = fmax(fabs(mu_new - mu), have_prev_pt ? fabs(mu - mu_prev) : 0.0);
      if (fabs(f) * st * inv_kT <= 2e-15 * C.Ne) { mu = mu_new; f = 0.0; done = true; break; }
    }
    mu_prev = mu; f_prev = f; have_prev_pt = true;
    mu = mu_new;
  }
  if ((sc_is_block_local || blockIdx.x == 0) && threadIdx.x == 0) {
    sc->mu = mu; sc->mu_lo = lo; sc->mu_hi = hi; sc->mu_evals = evals; sc->mu_evals_total += evals; sc->N_last = f + C.Ne;
  }
  return mu;   // identical in every thread of the grid
}

// First evaluation of the mu iteration as an ordinary (non-cooperative, programmatic-dependent) launch.  On mid-size
// grids the cooperative kernel below costs more in launch serialisation, table copies and grid barriers than in work
// (192^3: 52 us per evaluation against ~15 us of work; it also breaks the dependent-launch chain of the iteration), and
// in steady state the iteration needs exactly one evaluation: the verification of the Newton step taken from the fused
// evaluation of the S2 pass.  This kernel takes that step (same rules as mu_solve_dev: bracket, bisection when Newton
// leaves it), evaluates N(mu_1), and its last block decides: done (neutral to 1e-14 N_e, or the secant step passes the
// second-order bound) -> mu, bracket, counters are written and mu_done = 1, the cooperative kernel returns at once;
// not done -> (mu_1, sum I_1/2, slope) are handed over in the fields the cooperative kernel reads as "previous mu with a
// fused evaluation" and it carries on from there.  Streaming form of the evaluation only (even point count).
__global__ void __launch_bounds__(256, 3) mu_first_eval_kernel(const double *__restrict__ V_i, long long ng, ScfConst C,
                                                            DevScalars *sc, const double *__restrict__ fdtab,
                                                            double *partials, unsigned int *counter, const int *stop,
                                                            int final_try) {
  // final_try (the last of a chain of these launches that is NOT followed by the cooperative kernel): when the iteration
  // is still open at the end, the stop flag is set to 2 -- every later kernel of the batch returns at once and the host
  // finishes this SCF iteration with the cooperative kernel (arche.cu: scf_solve)
  extern __shared__ __align__(16) double s_tab[];
  __shared__ double s_red[64 + 2];
  __shared__ unsigned long long s_bar;
  pdl_launch_dependents();
  fd_load_tables_async(s_tab, fdtab, &s_bar);
  pdl_wait();
  if ((stop && *stop) || sc->mu_done) { fd_tables_wait(&s_bar); return; }   // uniform: written by earlier kernels only
  // the state every block derives for itself (sc is only written by the last block, after the grid reduction)
  const double inv_kT = 1.0 / C.kT, scaleN = C.cTF * C.dV;
  double lo = sc->mu_lo, hi = sc->mu_hi;
  const double mu0 = sc->mu, f0 = scaleN * sc->n0sum - C.Ne, slope0 = sc->dNdmu;
  const bool usable = sc->mu_have_prev && slope0 > 0.0 && !(hi - lo <= 4e-16 * fmax(fabs(lo), fabs(hi)));
  if (!usable) {                                             // first iteration / flat potential: the cooperative kernel
    if (final_try && stop && blockIdx.x == 0 && threadIdx.x == 0) sc->converged = 2;
    fd_tables_wait(&s_bar);
    return;
  }
  bool at_once = fabs(f0) <= 1e-14 * C.Ne;                   // the fused evaluation is already neutral
  double mu1 = mu0;
  if (!at_once) {
    if (f0 > 0.0) hi = fmin(hi, mu0); else lo = fmax(lo, mu0);
    mu1 = mu0 - f0 / slope0;
    if (!(mu1 > lo && mu1 < hi)) mu1 = 0.5 * (lo + hi);
    if (fabs(mu1 - mu0) <= 2e-16 * fmax(fabs(mu0), C.kT)) at_once = true;
  }
  if (at_once) {
    if (blockIdx.x == 0 && threadIdx.x == 0) {
      sc->mu_evals = 1; sc->mu_evals_total += 1; sc->N_last = f0 + C.Ne; sc->mu_done = 1;
    }
    fd_tables_wait(&s_bar);
    return;
  }
  fd_tables_wait(&s_bar);
  double s1 = 0.0;
  {
    const double sA = inv_kT * FD_INV_W, sB = (mu1 * inv_kT - FD_ETA_A) * FD_INV_W;   // s = sB - v sA
    const double2 *V2 = reinterpret_cast<const double2 *>(V_i);
    const int n2 = (int)(ng >> 1), nth = (int)(gridDim.x * blockDim.x);
    int i = (int)(blockIdx.x * blockDim.x + threadIdx.x);
    const double2 zero2 = make_double2(0.0, 0.0);
    double2 a = i < n2 ? V2[i] : zero2, b = i + nth < n2 ? V2[i + nth] : zero2;
    for (; i < n2; i += 2 * nth) {
      const int in = i + 2 * nth;
      const double2 an = in < n2 ? V2[in] : zero2, bn = in + nth < n2 ? V2[in + nth] : zero2;
      if (i + nth < n2) {
        const double sg[4] = {fma(-a.x, sA, sB), fma(-a.y, sA, sB), fma(-b.x, sA, sB), fma(-b.y, sA, sB)};
        double im12[4], i12[4], d[4];
        fd_eval_multi_s<2, 4>(s_tab, sg, im12, i12, d);
        s1 += (i12[0] + i12[1]) + (i12[2] + i12[3]);
      } else {
        const double sg[2] = {fma(-a.x, sA, sB), fma(-a.y, sA, sB)};
        double im12[2], i12[2], d[2];
        fd_eval_multi_s<2, 2>(s_tab, sg, im12, i12, d);
        s1 += i12[0] + i12[1];
      }
      a = an; b = bn;
    }
  }
  double v[1] = {s1};
  const int op[1] = {0};
  if (grid_reduce<1>(v, op, partials, counter, s_red) && threadIdx.x == 0) {
    const double S1 = s_red[32], f1 = scaleN * S1 - C.Ne;
    bool done = false;
    double mu = mu1, fres = f1, slope = slope0;
    if (fabs(f1) <= 1e-14 * C.Ne) done = true;
    else {
      if (f1 > 0.0) hi = fmin(hi, mu1); else lo = fmax(lo, mu1);
      bool fresh = false;
      if (mu1 != mu0) { const double sct = (f1 - f0) / (mu1 - mu0); if (sct > 0.0) { slope = sct; fresh = true; } }
      double mu2 = mu1 - f1 / slope;
      if (!(mu2 > lo && mu2 < hi)) mu2 = 0.5 * (lo + hi);
      if (fabs(mu2 - mu1) <= 2e-16 * fmax(fabs(mu1), C.kT)) done = true;
      else if (fresh) {
        const double st = fmax(fabs(mu2 - mu1), fabs(mu1 - mu0));
        if (fabs(f1) * st * inv_kT <= 2e-15 * C.Ne) { mu = mu2; fres = 0.0; done = true; }
      }
    }
    sc->mu_lo = lo; sc->mu_hi = hi; sc->mu = mu;
    if (done) { sc->mu_evals = 2; sc->mu_evals_total += 2; sc->N_last = fres + C.Ne; sc->mu_done = 1; }
    else {   // hand-over: (mu_1, f_1) as the "fused" evaluation of whoever continues
      sc->n0sum = S1; sc->dNdmu = slope; sc->mu_evals_total += 1;
      if (final_try && stop) sc->converged = 2;
    }
  }
}

__global__ void __launch_bounds__(256, 3) mu_solve_kernel(const double *__restrict__ V_i, long long ng, ScfConst C,
                                                       DevScalars *sc, const double *__restrict__ fdtab,
                                                       double *partials, int max_pass, const int *stop) {
  namespace cg = cooperative_groups;
  if (stop && *stop) return;   // uniform over the grid: no block reaches a barrier
  if (sc->mu_done) return;     // mu_first_eval_kernel finished the iteration (uniform: written before this launch)
  cg::grid_group grid = cg::this_grid();
  extern __shared__ __align__(16) double s_tab[];   // kFdTabDoubles (49.5 KB: dynamic, beyond the 48 KB static limit)
  __shared__ double s_red[2 * 32 + 2];
  __shared__ double s_bc[2];
  __shared__ unsigned long long s_bar;
  fd_load_tables(s_tab, fdtab, &s_bar);
  mu_solve_dev(grid, V_i, ng, C, sc, s_tab, s_red, s_bc, partials, max_pass);
}

// ---- S4 fused into the forward x pass: n_a, chi and the local reductions K, ||dn||^2, ||n_a||^2, F0, K_e, E_xc,
// dN/dmu are formed while the real lines of n_a are loaded for the transform; n_a is also stored (mixing needs it).
struct LoadDensity {
  const double *V_i, *n_i;
  double *n_a;
  DevScalars *sc;
  double *partials;
  unsigned int *counter;
  const double *fdtab;
  ScfConst C;
  double mu, inv_kT, sK, sdn2, sna2, sF0, sKe, sExc, sChi;
  bool wantF;   // uniform: this iteration evaluates the free-energy terms (F_0, K_e, E_xc)
  __device__ __forceinline__ void set_table(const double *t) { fdtab = t; }
  __device__ __forceinline__ void begin() {
    mu = sc->mu; inv_kT = 1.0 / C.kT;
    sK = sdn2 = sna2 = sF0 = sKe = sExc = sChi = 0.0;
    wantF = sc->skip_F == 0;
  }
  __device__ __forceinline__ void prefetch(long long idx) const { prefetch_l2(V_i + idx); prefetch_l2(n_i + idx); }
  __device__ __forceinline__ double load_real(long long g, int, int, int) {
    const double eta = (mu - V_i[g]) * inv_kT;
    double im12, i12, i32 = 0.0;
    if (wantF) fd_eval<7>(fdtab, eta, im12, i12, i32); else fd_eval<3>(fdtab, eta, im12, i12, i32);
    const double na = C.cTF * i12;                    // Eq. 9
    const double chi = C.cTF * 0.5 * im12 * inv_kT;   // dn_a/dmu
    const double dn = n_i[g] - na;
    n_a[g] = na;
    if (chi > 1.0e-290) sK += dn * dn * rcp_fast(fmax(chi, C.chi_floor));   // Eq. 31 (reading A11c: optional lower bound)
    sdn2 += dn * dn; sna2 += na * na; sChi += chi;
    if (wantF) {
      sF0 += eta * i12 - (2.0 / 3.0) * i32;           // f_0/(kT cTF), from Eq. 38-39
      sKe += i32;                                     // Eq. 38
      if (C.xc) { double e, vx; xc_pz81(na, e, vx, C.xc); sExc += na * e; }
    }
    return na;
  }
  struct Pre { double v0, v1, n0, n1; };
  __device__ __forceinline__ void fetch(long long ia, long long ib, Pre &p) const {
    p.v0 = V_i[ia]; p.v1 = V_i[ib]; p.n0 = n_i[ia]; p.n1 = n_i[ib];
  }
  __device__ __forceinline__ void compute(long long ia, long long ib, const Pre &p, double &ra, double &rb) {
    const long long g[2] = {ia, ib};
    double eta[2] = {(mu - p.v0) * inv_kT, (mu - p.v1) * inv_kT}, im12[2], i12[2], i32[2] = {0.0, 0.0};
    const double ni[2] = {p.n0, p.n1};
    if (wantF) fd_eval_multi<7, 2>(fdtab, eta, im12, i12, i32); else fd_eval_multi<3, 2>(fdtab, eta, im12, i12, i32);
    double na[2];
#pragma unroll
    for (int m = 0; m < 2; ++m) {
      na[m] = C.cTF * i12[m];
      const double chi = C.cTF * 0.5 * im12[m] * inv_kT;
      const double dn = ni[m] - na[m];
      n_a[g[m]] = na[m];
      if (chi > 1.0e-290) sK += dn * dn * rcp_fast(fmax(chi, C.chi_floor));   // Eq. 31 (reading A11c: optional lower bound)
      sdn2 += dn * dn; sna2 += na[m] * na[m]; sChi += chi;
    }
    if (wantF) {
#pragma unroll
      for (int m = 0; m < 2; ++m) {
        sF0 += eta[m] * i12[m] - (2.0 / 3.0) * i32[m];
        sKe += i32[m];
        if (C.xc) { double e, vx; xc_pz81(na[m], e, vx, C.xc); sExc += na[m] * e; }
      }
    }
    ra = na[0]; rb = na[1];
  }
  __device__ __forceinline__ void load_real2(long long ia, long long ib, double &ra, double &rb) {
    Pre p; fetch(ia, ib, p); compute(ia, ib, p, ra, rb);
  }
  __device__ __forceinline__ void finish(double *smem) {
    double v[7] = {sK, sdn2, sna2, sF0, sKe, sExc, sChi};
    const int op[7] = {0, 0, 0, 0, 0, 0, 0};
    if (grid_reduce<7>(v, op, partials, counter, smem) && threadIdx.x == 0) apply(smem + 7 * 32, C, sc);
  }
  static __device__ __forceinline__ void apply(const double *t, const ScfConst &C, DevScalars *sc) {
    sc->K = t[0] * C.dV; sc->dn2 = t[1] * C.dV; sc->na2 = t[2] * C.dV;
    sc->F0 = t[3] * C.dV * C.kT * C.cTF; sc->Ke = t[4] * C.dV * C.kT * C.cTF; sc->Exc = t[5] * C.dV;
    sc->dNdmu = t[6] * C.dV;
  }
  __device__ __forceinline__ void partial(double *smem, double *out /*[gridDim.x][stride]*/, int stride = 7, int offset = 0) {
    double v[7] = {sK, sdn2, sna2, sF0, sKe, sExc, sChi};
    const int op[7] = {0, 0, 0, 0, 0, 0, 0};
    block_partials<7>(v, op, smem, out, stride, offset);
  }
};

// ---- S5: forward FFT of the real n_a; the z-pass epilogue scales by dV, stores nhat_a, reduces U, E_H, E_ie ------
struct LoadReal {
  const double *src;
  __device__ __forceinline__ void set_table(const double *) {}
  __device__ __forceinline__ void begin() {}
  __device__ __forceinline__ void prefetch(long long idx) const { prefetch_l2(src + idx); }
  __device__ __forceinline__ void operator()(long long idx, int, int, int, double &re, double &im) { re = src[idx]; im = 0.0; }
  __device__ __forceinline__ double load_real(long long idx, int, int, int) { return src[idx]; }
  __device__ __forceinline__ void load_real2(long long ia, long long ib, double &ra, double &rb) { ra = src[ia]; rb = src[ib]; }
  struct Pre { double a, b; };
  __device__ __forceinline__ void fetch(long long ia, long long ib, Pre &p) const { p.a = src[ia]; p.b = src[ib]; }
  __device__ __forceinline__ void compute(long long, long long, const Pre &p, double &ra, double &rb) { ra = p.a; rb = p.b; }
  __device__ __forceinline__ void finish(double *) {}
};

struct StoreNhatA {
  static constexpr bool kSplitStore = true;
  double2 *nh_a;
  const double2 *nh_i, *vh_ie;
  const double *kx2, *ky2, *kz2;
  DevScalars *sc;
  double *partials;
  unsigned int *counter;
  ScfConst C;
  HalfGeom H;
  int prestored;   // 1: the value is already scaled and stored in nh_a (streaming reduction after a plain z pass)
  double aU, aEH, aEie;
  bool wantF;   // uniform: this iteration evaluates E_ie (the only use of Vhat_ie in S5)
  __device__ __forceinline__ void begin() { aU = aEH = aEie = 0.0; wantF = sc->skip_F == 0; }
  __device__ __forceinline__ void prefetch(long long idx) const { if (wantF) prefetch_l2(vh_ie + idx); prefetch_l2(nh_i + idx); }
  __device__ __forceinline__ void store(long long idx, int ix, int iy, int iz, double re, double im) {
    if (ix >= H.nxh) { if (!prestored) nh_a[idx] = make_double2(0.0, 0.0); return; }
    if (!prestored) { re *= C.dV; im *= C.dV; nh_a[idx] = make_double2(re, im); }
    const double wt = H.wt(ix);
    if (wantF) { const double2 b = vh_ie[idx]; aEie += wt * (re * b.x + im * b.y); }   // Re conj(nhat_a) Vhat_ie
    const double k2 = kx2[ix] + ky2[iy] + kz2[iz];
    if (k2 != 0.0) {
      const double inv = wt * __drcp_rn(ARCHE_PI * k2);
      const double2 a = nh_i[idx];
      const double dr = a.x - re, di = a.y - im;
      aU += (dr * dr + di * di) * inv;                   // Eq. 30
      aEH += (re * re + im * im) * inv;                  // Eq. 53
    }
  }
  // split form of store(): accumulate() scales v in place and does every load and reduction, put() stores
  __device__ __forceinline__ void accumulate(long long idx, int ix, int iy, int iz, double2 &v) {
    if (ix >= H.nxh) { v = make_double2(0.0, 0.0); return; }
    v.x *= C.dV; v.y *= C.dV;
    const double wt = H.wt(ix);
    if (wantF) { const double2 b = vh_ie[idx]; aEie += wt * (v.x * b.x + v.y * b.y); }
    const double k2 = kx2[ix] + ky2[iy] + kz2[iz];
    if (k2 != 0.0) {
      const double inv = wt * __drcp_rn(ARCHE_PI * k2);
      const double2 a = nh_i[idx];
      const double dr = a.x - v.x, di = a.y - v.y;
      aU += (dr * dr + di * di) * inv;
      aEH += (v.x * v.x + v.y * v.y) * inv;
    }
  }
  __device__ __forceinline__ void put(long long idx, double2 v) { nh_a[idx] = v; }
  __device__ __forceinline__ void finish(double *smem) {
    double v[3] = {aU, aEH, aEie};
    const int op[3] = {0, 0, 0};
    if (grid_reduce<3>(v, op, partials, counter, smem) && threadIdx.x == 0) apply(smem + 3 * 32, C, sc);
  }
  __device__ __forceinline__ void partial(double *smem, double *out /*[gridDim.x][stride]*/, int stride = 3, int offset = 0) {
    double v[3] = {aU, aEH, aEie};
    const int op[3] = {0, 0, 0};
    block_partials<3>(v, op, smem, out, stride, offset);
  }
  // grid totals {U, E_H, E_ie sums} -> energies, w (Eq. 30-31), free energy and the stop flag
  static __device__ __forceinline__ void apply(const double *t, const ScfConst &C, DevScalars *sc) {
    {
      const double U = t[0] * C.inv_vol, EH = 0.5 * t[1] * C.inv_vol, Eie = t[2] * C.inv_vol;
      sc->U = U; sc->EH = EH; sc->Eie = Eie;
      const int it = sc->iter + 1;
      const double K = sc->K;
      // reading A11b ("w is computed and updated only after a few SCF iterations, once the chemical potential
      // fluctuations are small"): after the warm-up count, and -- when mix_mu_tol > 0 -- once two successive mu_a differ
      // by at most mix_mu_tol kT; the switch is latched for the rest of the solve
      // the fluctuation is measured per unit of undamped step: the input moved by (1 - w_prev)(n_a - n_i) since the last
      // iteration, so |mu_k - mu_{k-1}|/(1 - w_prev) estimates what a full step would do to mu (with w_prev = 0.99 two
      // successive mu agree to 1e-3 kT by construction, however far the density is from the fixed point)
      if (C.mix_mu_tol > 0.0 && !sc->more_on && it >= 2 &&
          fabs(sc->mu - sc->mu_iter_prev) <= C.mix_mu_tol * C.kT * (1.0 - sc->w)) sc->more_on = 1;
      sc->mu_iter_prev = sc->mu;
      double w;
      if (C.mix_mode == 1 && it > C.mix_warmup && (C.mix_mu_tol <= 0.0 || sc->more_on)) w = (K + U > 0.0) ? U / (K + U) : 0.0;   // w = U/(K+U)
      else w = C.mix_w_fixed;
      const bool haveF = sc->skip_F == 0;   // this iteration evaluated F0, E_xc, E_ie (always, unless C.lazy_F)
      const double F = haveF ? sc->F0 + sc->Exc + EH + Eie + C.E_ie0 + sc->U_ii : sc->F_total;
      const double dn_rel = sqrt(sc->dn2 / sc->na2);
      // reading A13: PZ81's two branches differ by 3.2e-5 Ha (eps_c) / 2.7e-5 Ha (V_c) at r_s = 1, n* = 3/(4 pi).  A grid
      // point whose converged density sits on n* flips branch between iterations: F then moves by whole quanta
      // q_F = (eps_c jump) n* dV and the density answers the V_c jump with a limit cycle of relative size
      // q_dn/||n_a|| -- neither criterion can be met below that.  A jump of F by an integer number (1..8) of quanta
      // marks the solve; from then on two quanta are tolerated in both criteria.  flip_seen and the tolerances applied
      // are reported in arche_result.
      const double dFs = F - sc->F_total, dF = (haveF && (sc->F_valid || !C.lazy_F)) ? fabs(dFs) : 1.0e300;
      if (C.xc == 1 && it >= 3 && C.q_F > 0.0) {
        const double dFp = sc->F_total - sc->F_prev;
        const double m = dF * C.inv_qF, r = rint(m), mp = fabs(dFp) * C.inv_qF, rp = rint(mp);
        const bool near = r >= 1.0 && r <= 8.0 && fabs(m - r) < 0.02, near_prev = rp >= 1.0 && rp <= 8.0 && fabs(mp - rp) < 0.02;
        // (a) a quantised jump right after a change far below one quantum, or (b) the same multiple twice in a row with
        // opposite signs (F hops back: a flip that set in before F had settled).  The free energy of a converging solve
        // decreases monotonically -- also a slowly converging one, whose successive dF are nearly equal -- so (b) cannot
        // fire on a smooth decay.
        if (near && (mp < 0.1 || (near_prev && r == rp && dFs * dFp < 0.0))) sc->flip_seen = 1;
      }
      const double tolF = C.tol_F + (sc->flip_seen ? 2.02 * C.q_F : 0.0);
      const double toldn = C.tol_dn + (sc->flip_seen ? 2.0 * C.q_dn / sqrt(sc->na2) : 0.0);
      sc->converged = (it >= 2 && dF < tolF && dn_rel < toldn) ? 1 : 0;
      sc->tolF_eff = tolF; sc->toldn_eff = toldn;
      if (C.lazy_F > 0) {
        // F is needed in the iteration that meets the density criterion and in the one before it: predict the residual
        // two iterations ahead from the last contraction factor (a wrong guess costs iterations, never the result)
        const double rho = (it >= 2 && sc->dn_rel > 0.0) ? fmin(fmax(dn_rel / sc->dn_rel, 0.05), 1.0) : 1.0;
        sc->skip_F = (dn_rel * rho * rho > 4.0 * toldn && it + 1 < C.lazy_F) ? 1 : 0;
      }
      sc->F_valid = haveF ? 1 : 0;
      if (haveF) sc->F_evals += 1;
      if (haveF) sc->F_prev = sc->F_total;
      sc->F_total = F; sc->w = w; sc->dn_rel = dn_rel; sc->iter = it;
      sc->mu_have_prev = 1;
    }
  }
};

// ---- S6: n_o = n_a + w (n_i - n_a) in real and reciprocal space.  Inside the SCF loop this is fused into
// the next iteration's S1/S2 passes; this kernel materialises a pending step when n_i is read back.
__global__ void __launch_bounds__(256) mix_kernel(double *__restrict__ n_i, const double *__restrict__ n_a,
                                                  double2 *__restrict__ nh_i, const double2 *__restrict__ nh_a,
                                                  long long ng, long long nh, const DevScalars *sc) {
  const double w = sc->w;
  const long long stride = (long long)gridDim.x * blockDim.x, t0 = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  for (long long g = t0; g < ng; g += stride) {
    const double na = n_a[g];
    n_i[g] = fma(w, n_i[g] - na, na);
  }
  for (long long g = t0; g < nh; g += stride) {
    const double2 a = nh_a[g], b = nh_i[g];
    nh_i[g] = make_double2(fma(w, b.x - a.x, a.x), fma(w, b.y - a.y, a.y));
  }
}

// ---- input density: uniform or one-center profile (reading A10) ------------------------
__global__ void set_uniform_kernel(double *n_i, double2 *nh_i, long long ng, long long nh, double n0, double Ne) {
  const long long stride = (long long)gridDim.x * blockDim.x, t0 = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  for (long long g = t0; g < ng; g += stride) n_i[g] = n0;
  for (long long g = t0; g < nh; g += stride) nh_i[g] = make_double2(g == 0 ? Ne : 0.0, 0.0);
}

// ghat = nhat_a conj(S)/max(|S|^2, eps Q^2) and the same with the Nyquist-flipped S2 (ion_kernels.cuh)
__global__ void g_store_kernel(double2 *__restrict__ gh, double2 *__restrict__ gh2, const double2 *__restrict__ nh_a,
                               const double2 *__restrict__ S, const double2 *__restrict__ S2, long long nh, double epsS) {
  for (long long g = (long long)blockIdx.x * blockDim.x + threadIdx.x; g < nh; g += (long long)gridDim.x * blockDim.x) {
    const double2 a = nh_a[g];
    double2 s = S[g];
    double inv = 1.0 / fmax(s.x * s.x + s.y * s.y, epsS);
    gh[g] = make_double2((a.x * s.x + a.y * s.y) * inv, (a.y * s.x - a.x * s.y) * inv);
    s = S2[g];
    inv = 1.0 / fmax(s.x * s.x + s.y * s.y, epsS);
    gh2[g] = make_double2((a.x * s.x + a.y * s.y) * inv, (a.y * s.x - a.x * s.y) * inv);
  }
}

// nhat_i = S_Z^{new} ghat^{old} (Eq. 20) symmetrised so that the half-spectrum inverse returns the real part of the
// full inverse transform (reading A6): X_sym = (S ghat + S2 ghat2)/2, equal to S ghat off the Nyquist planes.
struct LoadSG {
  static constexpr bool kWriteBack = false;
  const double2 *S, *S2, *gh, *gh2;
  int nxh;
  __device__ __forceinline__ void begin() {}
  __device__ __forceinline__ void prefetch(long long idx) const {
    prefetch_l2(S + idx); prefetch_l2(S2 + idx); prefetch_l2(gh + idx); prefetch_l2(gh2 + idx);
  }
  __device__ __forceinline__ void operator()(long long idx, int ix, int, int, double &re, double &im) {
    if (ix >= nxh) { re = 0.0; im = 0.0; return; }
    const double2 s = S[idx], g = gh[idx], s2 = S2[idx], g2 = gh2[idx];
    re = 0.5 * ((s.x * g.x - s.y * g.y) + (s2.x * g2.x - s2.y * g2.y));
    im = 0.5 * ((s.x * g.y + s.y * g.x) + (s2.x * g2.y + s2.y * g2.x));
  }
  __device__ __forceinline__ void finish(double *) {}
};

struct StoreClip {  // n_i = max(IFFT/|Omega|, floor), accumulates sum n_i
  double *n_i;
  DevScalars *sc;
  double *partials;
  unsigned int *counter;
  double inv_vol, floor_n, Ne, dV, acc;
  __device__ __forceinline__ void begin() { acc = 0.0; }
  __device__ __forceinline__ void prefetch(long long) const {}
  __device__ __forceinline__ void store_real(long long idx, int, int, int, double re) {
    double v = fmax(re * inv_vol, floor_n);
    n_i[idx] = v; acc += v;
  }
  __device__ __forceinline__ void store_real2(long long ia, long long ib, double ra, double rb) {
    store_real(ia, 0, 0, 0, ra); store_real(ib, 0, 0, 0, rb);
  }
  __device__ __forceinline__ void finish(double *smem) {
    double v[1] = {acc};
    const int op[1] = {0};
    if (grid_reduce<1>(v, op, partials, counter, smem) && threadIdx.x == 0) {
      sc->init_sum = smem[32] * dV;
      sc->init_scale = Ne / (smem[32] * dV);
    }
  }
};

struct LoadRealScaled {  // reads n_i, rescales to N_e, writes it back and feeds the forward FFT
  double *n_i;
  const DevScalars *sc;
  double scale;
  __device__ __forceinline__ void begin() { scale = sc->init_scale; }
  __device__ __forceinline__ void prefetch(long long idx) const { prefetch_l2(n_i + idx); }
  __device__ __forceinline__ double load_real(long long idx, int, int, int) {
    const double v = n_i[idx] * scale;
    n_i[idx] = v;
    return v;
  }
  __device__ __forceinline__ void load_real2(long long ia, long long ib, double &ra, double &rb) {
    ra = load_real(ia, 0, 0, 0); rb = load_real(ib, 0, 0, 0);
  }
  __device__ __forceinline__ void finish(double *) {}
};

struct StoreScaled {  // half spectrum, scaled; zero in the padding columns
  static constexpr bool kSplitStore = false;
  double2 *dst;
  double scale;
  int nxh;
  __device__ __forceinline__ void begin() {}
  __device__ __forceinline__ void prefetch(long long) const {}
  __device__ __forceinline__ void store(long long idx, int ix, int, int, double re, double im) {
    dst[idx] = ix < nxh ? make_double2(re * scale, im * scale) : make_double2(0.0, 0.0);
  }
  __device__ __forceinline__ void finish(double *) {}
};

struct StoreRealPlain {
  double *dst;
  __device__ __forceinline__ void begin() {}
  __device__ __forceinline__ void prefetch(long long) const {}
  __device__ __forceinline__ void store_real(long long idx, int, int, int, double v) { dst[idx] = v; }
  __device__ __forceinline__ void store_real2(long long ia, long long ib, double ra, double rb) { dst[ia] = ra; dst[ib] = rb; }
  __device__ __forceinline__ void finish(double *) {}
};

// ---- streaming forms of the pointwise work (large grids) -----------------------------------------------------
// On grids beyond the L2 the fused prologues/epilogues above run inside FFT tiles at two blocks per SM, which is too
// little parallelism for their extra operand streams (z passes) and their Fermi-Dirac/XC arithmetic (x passes).
// There the same functors run in these grid-stride kernels at full occupancy, around plain FFT passes.
struct StoreNull {
  __device__ __forceinline__ void set_table(const double *) {}
  __device__ __forceinline__ void begin() {}
  __device__ __forceinline__ void prefetch(long long) const {}
  __device__ __forceinline__ void store_real2(long long, long long, double, double) {}
  struct Pre {};
  __device__ __forceinline__ void fetch(long long, long long, Pre &) const {}
  __device__ __forceinline__ void compute(long long, long long, const Pre &, double, double) {}
  __device__ __forceinline__ void finish(double *) {}
};

template <class LoadOp, class StoreOp>
__global__ void __launch_bounds__(256) pointwise_g_kernel(LoadOp ld_in, StoreOp st_in, int P, int ny, long long nh,
                                                          const int *stop) {
  __shared__ double s_red[kMaxRed * 33];
  pdl_launch_dependents();
  pdl_wait();
  if (stop && *stop) return;
  LoadOp ld = ld_in;
  StoreOp st = st_in;
  ld.begin(); st.begin();
  for (long long h = (long long)blockIdx.x * blockDim.x + threadIdx.x; h < nh; h += (long long)gridDim.x * blockDim.x) {
    const int ix = (int)(h % P);
    const long long row = h / P;
    double re, im;
    ld(h, ix, (int)(row % ny), (int)(row / ny), re, im);
    st.store(h, ix, (int)(row % ny), (int)(row / ny), re, im);
  }
  ld.finish(s_red);
  st.finish(s_red);
}

// S5 reduction of the streamed form as a row walk (round 2).  ncu of pointwise_g_kernel<LoadComplex, StoreNhatA> at
// 384^3: 3.4 TB/s where a plain reduction of the same bytes reaches 6.9 TB/s on this GPU -- one element per thread and
// step, four 64-bit divisions per element to recover (ix, iy, iz), long_scoreboard 13 warps per issue.  Here a thread
// keeps its column: kx^2 and the half-spectrum weight are registers, a block walks over a contiguous range of (ky, kz)
// rows and carries (iy, iz) along, four rows -- eight or twelve 16-byte loads per thread -- are in flight at a time, and
// the only per-element arithmetic left is the reciprocal of pi k^2.  Same sums, same closing step (StoreNhatA::finish).
template <int ROWS>
__global__ void __launch_bounds__(256) s5_rows_kernel(StoreNhatA st_in, int P, int ny, int nrows, int rows_per_block, const int *stop) {
  __shared__ double s_red[kMaxRed * 33];
  pdl_launch_dependents();
  pdl_wait();
  if (stop && *stop) return;
  StoreNhatA st = st_in;
  st.begin();
  const int r0 = blockIdx.x * rows_per_block, r1 = min(nrows, r0 + rows_per_block);
  for (int ix = threadIdx.x; ix < st.H.nxh; ix += blockDim.x) {
    const double kx2 = st.kx2[ix], wt = st.H.wt(ix);
    int iy = r0 % ny, iz = r0 / ny;
    for (int r = r0; r < r1; r += ROWS) {
      double2 v[ROWS], a[ROWS], b[ROWS];
      double k2[ROWS];
#pragma unroll
      for (int q = 0; q < ROWS; ++q) {
        const bool ok = r + q < r1;
        const long long h = (long long)(ok ? r + q : r) * P + ix;
        v[q] = st.nh_a[h]; a[q] = st.nh_i[h];
        if (st.wantF) b[q] = st.vh_ie[h];
        k2[q] = ok ? kx2 + st.ky2[iy] + st.kz2[iz] : 0.0;   // a row past the end counts like k = 0: nothing
        if (!ok) { v[q] = make_double2(0.0, 0.0); b[q] = v[q]; }
        if (++iy == ny) { iy = 0; ++iz; }
      }
#pragma unroll
      for (int q = 0; q < ROWS; ++q) {
        if (st.wantF) st.aEie += wt * (v[q].x * b[q].x + v[q].y * b[q].y);   // Re conj(nhat_a) Vhat_ie
        if (k2[q] != 0.0) {
          const double inv = wt * __drcp_rn(ARCHE_PI * k2[q]);
          const double dr = a[q].x - v[q].x, di = a[q].y - v[q].y;
          st.aU += (dr * dr + di * di) * inv;                              // Eq. 30
          st.aEH += (v[q].x * v[q].x + v[q].y * v[q].y) * inv;             // Eq. 53
        }
      }
    }
  }
  st.finish(s_red);
}

// real fields, two elements per thread and step (the functors interleave their two Fermi-Dirac evaluations); ng even.
// SMEM_TAB: the block first copies the Fermi-Dirac table (g_tab) to shared memory and the functors read it there --
// for the streamed form, launched with as many blocks as are co-resident (the table copy is paid once per block).
template <class LoadOp, class StoreOp, bool SMEM_TAB = false, int MIN_BLOCKS = 1>
__global__ void __launch_bounds__(256, MIN_BLOCKS) pointwise_r_kernel(LoadOp ld_in, StoreOp st_in, long long ng, const int *stop,
                                                          const double *__restrict__ g_tab = nullptr) {
  __shared__ double s_red[kMaxRed * 33];
  __shared__ unsigned long long s_bar;
  extern __shared__ __align__(16) double s_tab[];   // SMEM_TAB: kFdTabDoubles doubles of dynamic shared memory
  pdl_launch_dependents();
  if (SMEM_TAB) fd_load_tables_async(s_tab, g_tab, &s_bar);   // constant data: the copy runs while the predecessor drains
  pdl_wait();
  if (stop && *stop) {             // (the bulk copy must have landed before the block may exit)
    if (SMEM_TAB) fd_tables_wait(&s_bar);
    return;
  }
  LoadOp ld = ld_in;
  StoreOp st = st_in;
  if (SMEM_TAB) {
    fd_tables_wait(&s_bar);
    ld.set_table(s_tab); st.set_table(s_tab);
  }
  ld.begin(); st.begin();
  // software pipeline: the operands of the thread's next pair are loaded before it evaluates the current pair (ncu, round
  // 2: the first use of the loaded potentials was the hottest instruction of these kernels -- nothing else covered the
  // HBM latency at 24-32 warps per SM; an L2 prefetch hint instead of register loads made them slower)
  const long long half = ng / 2, stride = (long long)gridDim.x * blockDim.x;
  long long g = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  typename LoadOp::Pre pl, pln;
  typename StoreOp::Pre ps, psn;
  if (g < half) { ld.fetch(g, g + half, pl); st.fetch(g, g + half, ps); }
  for (; g < half; g += stride) {
    const long long gn = g + stride;
    if (gn < half) { ld.fetch(gn, gn + half, pln); st.fetch(gn, gn + half, psn); }
    double a, b;
    ld.compute(g, g + half, pl, a, b);
    st.compute(g, g + half, ps, a, b);
    pl = pln; ps = psn;
  }
  ld.finish(s_red);
  st.finish(s_red);
}

// Full-spectrum view [nz][ny][nx] of a half-spectrum array for read-back: ix <= nx/2 copies src, the rest is
// conj(src2[mirror]) (src2 = src for DFT-Hermitian fields, the Nyquist-flipped companion for S_Z and ghat);
// `scale` (optional, half-spectrum real array) multiplies the result (Vhat_ie = v(k) S_Z(k)).
__global__ void expand_half_kernel(double2 *__restrict__ dst, const double2 *__restrict__ src, const double2 *__restrict__ src2,
                                   const double *__restrict__ scale, int nx, int ny, int nz, int P) {
  const long long ng = (long long)nx * ny * nz;
  const int nxh = nx / 2 + 1;
  for (long long g = (long long)blockIdx.x * blockDim.x + threadIdx.x; g < ng; g += (long long)gridDim.x * blockDim.x) {
    const int ix = (int)(g % nx), iy = (int)((g / nx) % ny), iz = (int)(g / ((long long)nx * ny));
    double2 v;
    long long h;
    if (ix < nxh) { h = ((long long)iz * ny + iy) * P + ix; v = src[h]; }
    else {
      h = ((long long)((nz - iz) % nz) * ny + (ny - iy) % ny) * P + (nx - ix);
      v = src2[h]; v.y = -v.y;
    }
    if (scale) { const double sfac = scale[h]; v.x *= sfac; v.y *= sfac; }
    dst[g] = v;
  }
}

// half <- the stored columns of a full [nz][ny][nx] complex array (zero padding columns)
__global__ void compress_half_kernel(double2 *__restrict__ dst, const double2 *__restrict__ src, int nx, int ny, int nz, int P) {
  const long long nh = (long long)P * ny * nz;
  const int nxh = nx / 2 + 1;
  for (long long h = (long long)blockIdx.x * blockDim.x + threadIdx.x; h < nh; h += (long long)gridDim.x * blockDim.x) {
    const int ix = (int)(h % P);
    const long long row = h / P;
    dst[h] = ix < nxh ? src[row * nx + ix] : make_double2(0.0, 0.0);
  }
}

__global__ void fermi_dirac_kernel(int twice_j, const double *eta, double *out, size_t n, const double *fdtab) {
  extern __shared__ __align__(16) double s_tab[];   // kFdTabDoubles
  __shared__ unsigned long long s_bar;
  fd_load_tables(s_tab, fdtab, &s_bar);
  for (size_t g = (size_t)blockIdx.x * blockDim.x + threadIdx.x; g < n; g += (size_t)gridDim.x * blockDim.x) {
    double a, b, c;
    fd_eval<7>(s_tab, eta[g], a, b, c);
    out[g] = twice_j == -1 ? a : (twice_j == 1 ? b : c);
  }
}

}  // namespace arche
