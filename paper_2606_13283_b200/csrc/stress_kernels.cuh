// stress_kernels.cuh -- f1: average virial stress tensor and pressure of the converged state (PAPER.md:341-347,
// Eq. 34-35; terms: Eq. 37 :355, Eq. 39 :372, Eq. 48-51 :423-440, Eq. 54 :458-461, sigma^ie :483-487; LDA term and
// sign convention: DESIGN.md reading A21).  sigma_mn = (1/|Omega|) dE/d(eps_mn), P = -tr(Sigma)/3.
//
// One streaming pass over the half spectrum (nhat_a, S_Z, S2: 48 B per stored point) and over n_a (8 B per point)
// gathers 21 sums; a pair kernel gathers the six short-range Ewald sums; a single-block kernel adds the partials in a
// fixed order and assembles the 9 x 6 table + P.
//
// Half spectrum and the literal index set (reading A6): a stored point p = (ix, iy, iz) stands for itself and for its
// index mirror p' = (-ix, -iy, -iz) mod N.  Off the Nyquist planes k(p') = -k(p) and every summand T is even, so the
// pair contributes wt(ix) T(p).  On a Nyquist plane k(p') = -k''(p), k'' = k with the Nyquist components' signs
// flipped, and S_Z(k(p')) = conj(S2(p)) (S2 from structure_factor_nyquist_kernel), so in general the pair contributes
//   wt(ix)/2 [ T(k, S) + T(k'', S2) ],   k''_m k''_n = s_m s_n k_m k_n,  s = -1 on a Nyquist component,
// which is the same expression off the planes (S2 = S, s = +1).
#pragma once
#include "common.cuh"
#include "scf_kernels.cuh"

namespace arche {

constexpr int kStressSums = 21;   // 0 pm trace part, 1..6 pm kk, 7 ee trace part, 8..13 ee kk, 14..19 ie kk, 20 int n (eps_xc - v_xc)
constexpr int kStressThreads = 256;
constexpr int kStressOut = 55;    // 9 rows x 6 columns + P

__global__ void __launch_bounds__(kStressThreads) stress_fields_kernel(
    GridGeom G, const double2 *__restrict__ nh_a, const double2 *__restrict__ S, const double2 *__restrict__ S2,
    const double *__restrict__ n_a, int xc, double alpha, double rc, PspTable T, double *__restrict__ partials /*[grid][21]*/) {
  __shared__ double s_red[kStressSums * 32];
  double acc[kStressSums];
#pragma unroll
  for (int q = 0; q < kStressSums; ++q) acc[q] = 0.0;
  const unsigned int P = (unsigned int)G.P, ny = (unsigned int)G.ny;
  const int nyq_x = (G.nx % 2 == 0) ? G.nx / 2 : -1, nyq_y = (G.ny % 2 == 0) ? G.ny / 2 : -1, nyq_z = (G.nz % 2 == 0) ? G.nz / 2 : -1;
  const double pi2_a2 = ARCHE_PI * ARCHE_PI / (alpha * alpha), inv_pi = 1.0 / ARCHE_PI, two_rc = 2.0 * rc;
  const long long stride = (long long)gridDim.x * blockDim.x;
  for (long long g = (long long)blockIdx.x * blockDim.x + threadIdx.x; g < G.nh; g += stride) {
    const unsigned int ug = (unsigned int)g, ix = ug % P, row = ug / P, iy = row % ny, iz = row / ny;
    if ((int)ix >= G.nxh) continue;
    const double kx = G.kx[ix], ky = G.ky[iy], kz = G.kz[iz];
    const double k2 = kx * kx + ky * ky + kz * kz;
    if (k2 == 0.0) continue;
    const double2 n = nh_a[g], s1 = S[g], s2 = S2[g];
    const double ik = rsqrt(k2), ik2 = ik * ik, ka = k2 * ik;   // one reciprocal square root instead of sqrt + three divisions
    const double hw = ((int)ix == 0 || (int)ix == nyq_x) ? 0.5 : 1.0;   // wt(ix)/2
    const bool fx = (int)ix == nyq_x, fy = (int)iy == nyq_y, fz = (int)iz == nyq_z;
    const double sg[3] = {(fy != fz) ? -1.0 : 1.0, (fx != fz) ? -1.0 : 1.0, (fx != fy) ? -1.0 : 1.0};   // yz, xz, xy
    const double kk[6] = {kx * kx, ky * ky, kz * kz, ky * kz, kx * kz, kx * ky};
    // Eq. 50: V_alpha |S_Z|^2 [2 k_m k_n (pi^2/alpha^2 + 1/k^2) - delta]
    const double va = exp(-pi2_a2 * k2) * inv_pi * ik2;
    const double a1 = va * (s1.x * s1.x + s1.y * s1.y), a2 = va * (s2.x * s2.x + s2.y * s2.y), cpm = pi2_a2 + ik2;
    // Eq. 54: |nhat|^2/(pi k^2) [2 k_m k_n/k^2 - delta]
    const double e = (n.x * n.x + n.y * n.y) * inv_pi * ik2;
    // Re(nhat conj(S_Z)) v'(k) k_m k_n/|k|, v(k) = -cos(2 pi k rc)/(pi k^2)
    double dv_k;   // v'(k)/k
    if (T.on) {    // f2: derivative of the tabulated form factor, -1/(pi k^2) + Du(k)
      double du;
      psp_table_interp(T, ka, &du);
      dv_k = (2.0 * inv_pi * ik2 * ik + du) * ik;
    } else {
      double sn, cs;
      sincospi(two_rc * ka, &sn, &cs);
      dv_k = (2.0 * rc * sn * ik2 + 2.0 * cs * inv_pi * ik2 * ik) * ik;
    }
    const double b1 = dv_k * (n.x * s1.x + n.y * s1.y), b2 = dv_k * (n.x * s2.x + n.y * s2.y);
    acc[0] += hw * (a1 + a2);
    acc[7] += 2.0 * hw * e;
#pragma unroll
    for (int q = 0; q < 3; ++q) {
      acc[1 + q] += hw * (a1 + a2) * cpm * kk[q];
      acc[8 + q] += 2.0 * hw * e * ik2 * kk[q];
      acc[14 + q] += hw * (b1 + b2) * kk[q];
    }
#pragma unroll
    for (int q = 3; q < 6; ++q) {
      const double s = sg[q - 3];
      acc[1 + q] += hw * (a1 + s * a2) * cpm * kk[q];
      acc[8 + q] += hw * (1.0 + s) * e * ik2 * kk[q];
      acc[14 + q] += hw * (b1 + s * b2) * kk[q];
    }
  }
  if (xc)
    for (long long r = (long long)blockIdx.x * blockDim.x + threadIdx.x; r < G.ng; r += stride) {
      const double n = n_a[r];
      double ex, vx;
      xc_pz81(n, ex, vx, xc);
      acc[20] += n * (ex - vx);
    }
  int op[kStressSums];
#pragma unroll
  for (int q = 0; q < kStressSums; ++q) op[q] = 0;
  block_reduce<kStressSums>(acc, op, s_red);
  if (threadIdx.x == 0) {
#pragma unroll
    for (int q = 0; q < kStressSums; ++q) partials[(size_t)blockIdx.x * kStressSums + q] = acc[q];
  }
}

// Eq. 49 with the minimum-image convention of Eq. 41: block j sums its pairs (j, k != j), half weight each.
__global__ void __launch_bounds__(128) stress_pp_kernel(const double *__restrict__ pos, const double *__restrict__ Z, int nions,
                                                        double Lx, double Ly, double Lz, double alpha,
                                                        double *__restrict__ pp_part /*[nions][6]*/) {
  __shared__ double s_red[6 * 32];
  const int j = blockIdx.x;
  const double xj = pos[3 * j], yj = pos[3 * j + 1], zj = pos[3 * j + 2], zq = Z[j];
  const double two_a_sqrtpi = 2.0 * alpha * 0.56418958354775628695;
  double a[6] = {0, 0, 0, 0, 0, 0};
  for (int k = threadIdx.x; k < nions; k += blockDim.x) {
    if (k == j) continue;
    double dx = xj - pos[3 * k], dy = yj - pos[3 * k + 1], dz = zj - pos[3 * k + 2];
    dx -= Lx * rint(dx / Lx); dy -= Ly * rint(dy / Ly); dz -= Lz * rint(dz / Lz);
    const double r2 = dx * dx + dy * dy + dz * dz, r = sqrt(r2);
    const double f = 0.5 * zq * Z[k] * (erfc(alpha * r) / r + two_a_sqrtpi * exp(-alpha * alpha * r2)) / r2;
    a[0] += f * dx * dx; a[1] += f * dy * dy; a[2] += f * dz * dz;
    a[3] += f * dy * dz; a[4] += f * dx * dz; a[5] += f * dx * dy;
  }
  const int op[6] = {0, 0, 0, 0, 0, 0};
  block_reduce<6>(a, op, s_red);
  if (threadIdx.x == 0) {
#pragma unroll
    for (int q = 0; q < 6; ++q) pp_part[6 * j + q] = a[q];
  }
}

struct StressConst {
  double vol, dV, alpha, Q, E_ie0;
};

// one block: fixed-order sums of the partials, then the table.  rows: i, e, xc, pp, pm, je, ee, ie, total
__global__ void __launch_bounds__(kStressThreads) stress_finish_kernel(int nblocks, const double *__restrict__ partials, int nions,
                                                                       const double *__restrict__ pp_part,
                                                                       const double *__restrict__ vel /*may be null*/,
                                                                       const double *__restrict__ mass, const DevScalars *sc,
                                                                       StressConst K, double *__restrict__ out /*[55]*/) {
  __shared__ double s_red[kStressSums * 32];
  __shared__ double s_f[kStressSums], s_pp[6], s_ki[6];
  {
    double acc[kStressSums];
    int op[kStressSums];
#pragma unroll
    for (int q = 0; q < kStressSums; ++q) { acc[q] = 0.0; op[q] = 0; }
    for (int b = threadIdx.x; b < nblocks; b += blockDim.x) {
#pragma unroll
      for (int q = 0; q < kStressSums; ++q) acc[q] += partials[(size_t)b * kStressSums + q];
    }
    block_reduce<kStressSums>(acc, op, s_red);
    if (threadIdx.x == 0) {
#pragma unroll
      for (int q = 0; q < kStressSums; ++q) s_f[q] = acc[q];
    }
  }
  {
    double a[6] = {0, 0, 0, 0, 0, 0}, b[6] = {0, 0, 0, 0, 0, 0};
    for (int j = threadIdx.x; j < nions; j += blockDim.x) {
#pragma unroll
      for (int q = 0; q < 6; ++q) a[q] += pp_part[6 * j + q];
      if (vel) {   // Eq. 37: m v_m v_n
        const double m = mass[j], vx = vel[3 * j], vy = vel[3 * j + 1], vz = vel[3 * j + 2];
        b[0] += m * vx * vx; b[1] += m * vy * vy; b[2] += m * vz * vz;
        b[3] += m * vy * vz; b[4] += m * vx * vz; b[5] += m * vx * vy;
      }
    }
    const int op[6] = {0, 0, 0, 0, 0, 0};
    block_reduce<6>(a, op, s_red);
    block_reduce<6>(b, op, s_red);
    if (threadIdx.x == 0) {
#pragma unroll
      for (int q = 0; q < 6; ++q) { s_pp[q] = a[q]; s_ki[q] = b[q]; }
    }
  }
  __syncthreads();
  if (threadIdx.x == 0) {
    const double vol = K.vol, iv2 = 1.0 / (vol * vol);
    double tot[6];
    for (int q = 0; q < 6; ++q) {
      const double dl = q < 3 ? 1.0 : 0.0;
      double r[8];
      r[0] = -s_ki[q] / vol;                                              // Eq. 37
      r[1] = -dl * 2.0 * sc->Ke / (3.0 * vol);                            // Eq. 39
      r[2] = dl * s_f[20] * K.dV / vol;                                   // reading A21
      r[3] = -s_pp[q] / vol;                                              // Eq. 49
      r[4] = (2.0 * s_f[1 + q] - dl * s_f[0]) * 0.5 * iv2;                // Eq. 50
      r[5] = dl * ARCHE_PI * K.Q * K.Q / (2.0 * K.alpha * K.alpha) * iv2; // Eq. 51
      r[6] = (2.0 * s_f[8 + q] - dl * s_f[7]) * 0.5 * iv2;                // Eq. 54
      r[7] = -s_f[14 + q] * iv2 - dl * (sc->Eie + K.E_ie0) / vol;         // P:483-487 with E^ie of Eq. 55
      double t = 0.0;
      for (int k = 0; k < 8; ++k) { out[6 * k + q] = r[k]; t += r[k]; }
      out[48 + q] = t;
      tot[q] = t;
    }
    out[54] = -(tot[0] + tot[1] + tot[2]) / 3.0;                          // Eq. 34
  }
}

}  // namespace arche
