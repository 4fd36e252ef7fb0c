// ion_kernels.cuh -- per-MD-step ion-grid work: separable phase tables, structure factor S_Z(k),
// ionic potential, Ewald, G-space forces, velocity Verlet.
// The O(N_i N_g) sums are tiled through shared memory and run on the fp64 FMA pipe (not tensor-core work).
#pragma once
#include "common.cuh"
#include "scf_kernels.cuh"

namespace arche {

// exp(-2 pi i m(i) x_j / L) for every storage index i of one axis and every ion j.
// tab_ij: [i][j] (j fastest); tab_ji: [j][i] (i fastest, optional).
__global__ void phase_table_kernel(const double *__restrict__ pos, int comp, double L, int N, int nions,
                                   double2 *__restrict__ tab_ij, double2 *__restrict__ tab_ji) {
  const long long tot = (long long)N * nions;
  for (long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x; e < tot; e += (long long)gridDim.x * blockDim.x) {
    const int j = (int)(e % nions), i = (int)(e / nions);
    const int m = i <= N / 2 ? i : i - N;
    double f = pos[3 * j + comp] / L;
    f -= floor(f);
    double t = (double)m * f;
    t -= rint(t);
    double s, c;
    sincospi(-2.0 * t, &s, &c);
    tab_ij[e] = make_double2(c, s);
    if (tab_ji) tab_ji[(long long)j * N + i] = make_double2(c, s);
  }
}

// f2: tabulated local pseudopotential.  u(k) = -1/(pi k^2) + Du(k) per unit charge; Du on the uniform grid
// k_m = m dk, cubic Lagrange polynomial through the nodes m0..m0+3, m0 = clamp(floor(k/dk) - 1, 0, nk - 4)
// (reading A22).  Returns Du(k); *du_dk (optional) the derivative of that cubic.
struct PspTable { int on, nk; double dk; const double *tab; };
__device__ __forceinline__ double psp_table_interp(const PspTable &T, double k, double *du_dk) {
  const double s = k / T.dk;
  int m0 = (int)floor(s) - 1;
  m0 = max(0, min(m0, T.nk - 4));
  const double t = s - (double)m0, y0 = T.tab[m0], y1 = T.tab[m0 + 1], y2 = T.tab[m0 + 2], y3 = T.tab[m0 + 3];
  const double t1 = t - 1.0, t2 = t - 2.0, t3 = t - 3.0;
  if (du_dk) {
    const double d0 = -(t2 * t3 + t1 * t3 + t1 * t2) * (1.0 / 6.0), d1 = (t2 * t3 + t * t3 + t * t2) * 0.5;
    const double d2 = -(t1 * t3 + t * t3 + t * t1) * 0.5, d3 = (t1 * t2 + t * t2 + t * t1) * (1.0 / 6.0);
    *du_dk = (y0 * d0 + y1 * d1 + y2 * d2 + y3 * d3) / T.dk;
  }
  return y0 * (-t1 * t2 * t3 * (1.0 / 6.0)) + y1 * (t * t2 * t3 * 0.5) + y2 * (-t * t1 * t3 * 0.5) + y3 * (t * t1 * t2 * (1.0 / 6.0));
}

// reciprocal-space form factors that depend only on the cell, on the half spectrum [nz][ny][P]: the pseudopotential per
// unit charge -- Ashcroft v(k) = -cos(2 pi k rc)/(pi k^2) or the tabulated one (f2) --, 0 at k = 0, and the
// Ewald kernel V_alpha(k) = exp(-(pi k/alpha)^2)/(pi k^2) (Eq. 43).  Zero in the padding columns.
__global__ void form_factor_kernel(GridGeom G, double rc, PspTable T, double alpha, double *__restrict__ vps, double *__restrict__ va) {
  const long long nh = (long long)G.P * G.ny * G.nz;
  for (long long g = (long long)blockIdx.x * blockDim.x + threadIdx.x; g < nh; g += (long long)gridDim.x * blockDim.x) {
    const int ix = (int)(g % G.P), iy = (int)((g / G.P) % G.ny), iz = (int)(g / ((long long)G.P * G.ny));
    if (ix >= G.nxh) { vps[g] = 0.0; va[g] = 0.0; continue; }
    const double k2 = G.kx2[ix] + G.ky2[iy] + G.kz2[iz];
    if (k2 == 0.0) { vps[g] = 0.0; va[g] = 0.0; continue; }
    const double k = sqrt(k2);
    vps[g] = T.on ? -1.0 / (ARCHE_PI * k2) + psp_table_interp(T, k, nullptr) : -cospi(2.0 * k * rc) / (ARCHE_PI * k2);
    va[g] = exp(-ARCHE_PI * ARCHE_PI * k2 / (alpha * alpha)) / (ARCHE_PI * k2);
  }
}

// S_Z(k) = sum_j Z_j a_j(kx) b_j(ky) c_j(kz) on the half spectrum.  A block owns SF_ROWS (ky,kz) rows and a chunk of
// kx; the ion sum is tiled: d_j = Z_j b_j c_j for SF_JT ions of every row is staged in shared memory, a_j(kx)
// streams coalesced.  Epilogue: Vhat_ie = v(k) S (Eq. 14) and the Ewald reciprocal energy sum of Eq. 42 with the
// half-spectrum weights; S2 = S (the Nyquist planes are corrected by structure_factor_nyquist_kernel).
constexpr int SF_ROWS = 4;
constexpr int SF_JT = 128;
constexpr int SF_THREADS = 128;
__global__ void __launch_bounds__(SF_THREADS) structure_factor_kernel(
    GridGeom G, int nions, const double *__restrict__ Z, const double2 *__restrict__ ax_ji /*[j][ix]*/,
    const double2 *__restrict__ by_ij /*[iy][j]*/, const double2 *__restrict__ cz_ij /*[iz][j]*/,
    const double *__restrict__ vps, const double *__restrict__ va, double2 *__restrict__ S, double2 *__restrict__ S2,
    double2 *__restrict__ vh_ie, double *partials, unsigned int *counter, DevScalars *sc) {
  __shared__ double2 s_d[SF_ROWS][SF_JT];
  __shared__ double s_red[32 + 1];
  const long long nrows = (long long)G.ny * G.nz;
  const long long row0 = (long long)blockIdx.x * SF_ROWS;
  const int ix = blockIdx.y * SF_THREADS + threadIdx.x;
  double2 acc[SF_ROWS];
#pragma unroll
  for (int r = 0; r < SF_ROWS; ++r) acc[r] = make_double2(0.0, 0.0);
  for (int j0 = 0; j0 < nions; j0 += SF_JT) {
    __syncthreads();
    for (int e = threadIdx.x; e < SF_ROWS * SF_JT; e += SF_THREADS) {
      const int r = e / SF_JT, jj = e % SF_JT, j = j0 + jj;
      const long long row = row0 + r;
      double2 d = make_double2(0.0, 0.0);
      if (j < nions && row < nrows) {
        const int iy = (int)(row % G.ny), iz = (int)(row / G.ny);
        const double2 b = by_ij[(long long)iy * nions + j], c = cz_ij[(long long)iz * nions + j];
        const double z = Z[j];
        d = make_double2(z * (b.x * c.x - b.y * c.y), z * (b.x * c.y + b.y * c.x));
      }
      s_d[r][jj] = d;
    }
    __syncthreads();
    if (ix < G.nxh) {
      const int jn = min(SF_JT, nions - j0);
      for (int jj = 0; jj < jn; ++jj) {
        const double2 a = ax_ji[(long long)(j0 + jj) * G.nx + ix];
#pragma unroll
        for (int r = 0; r < SF_ROWS; ++r) {
          const double2 d = s_d[r][jj];
          acc[r].x = fma(a.x, d.x, fma(-a.y, d.y, acc[r].x));
          acc[r].y = fma(a.x, d.y, fma(a.y, d.x, acc[r].y));
        }
      }
    }
  }
  double epm = 0.0;
  if (ix < G.P) {
    const double wt = (ix == 0 || 2 * ix == G.nx) ? 1.0 : 2.0;
#pragma unroll
    for (int r = 0; r < SF_ROWS; ++r) {
      const long long row = row0 + r;
      if (row < nrows) {
        const long long g = row * G.P + ix;
        if (ix < G.nxh) {
          S[g] = acc[r]; S2[g] = acc[r];
          const double v = vps[g];
          vh_ie[g] = make_double2(v * acc[r].x, v * acc[r].y);
          epm += wt * va[g] * (acc[r].x * acc[r].x + acc[r].y * acc[r].y);
        } else {
          S[g] = make_double2(0.0, 0.0); S2[g] = make_double2(0.0, 0.0); vh_ie[g] = make_double2(0.0, 0.0);
        }
      }
    }
  }
  // deterministic grid sum of the Ewald reciprocal term (2D grid flattened)
  double v[1] = {epm};
  const int op[1] = {0};
  block_reduce<1>(v, op, s_red);
  __shared__ bool s_last;
  const unsigned int nblk = gridDim.x * gridDim.y, bid = blockIdx.y * gridDim.x + blockIdx.x;
  if (threadIdx.x == 0) {
    partials[bid] = v[0];
    __threadfence();
    s_last = (atomicAdd(counter, 1u) == nblk - 1);
  }
  __syncthreads();
  if (s_last) {
    __threadfence();
    double a = 0.0;
    for (unsigned int b = threadIdx.x; b < nblk; b += blockDim.x) a += __ldcg(&partials[b]);
    double w[1] = {a};
    block_reduce<1>(w, op, s_red);
    if (threadIdx.x == 0) { sc->U_pm_sum = w[0]; *counter = 0u; }
  }
}

// Register-tiled form for the production grids (nx even, nx/2 a multiple of 32*IXT): every thread owns IXT kx columns x
// 8 (ky,kz) rows, so that one a_j(kx) word feeds 8 products and one staged d_j word IXT products -- the kernel above
// (1 column x 4 rows per thread) is bound by its broadcast shared-memory reads at 0.46 of the fp64 peak.  Covers
// kx < nx/2; the column kx = nx/2 is left to structure_factor_nyquist_kernel (all of it lies on a Nyquist plane),
// the padding columns stay zero from arche_scf_init.
constexpr int SF2_ROWS = 8;
constexpr int SF2_JT = 64;
template <int IXT>
__global__ void __launch_bounds__(256) structure_factor_tiled_kernel(
    GridGeom G, int nions, const double *__restrict__ Z, const double2 *__restrict__ ax_ji /*[j][ix]*/,
    const double2 *__restrict__ by_ij /*[iy][j]*/, const double2 *__restrict__ cz_ij /*[iz][j]*/,
    const double *__restrict__ vps, const double *__restrict__ va, double2 *__restrict__ S, double2 *__restrict__ S2,
    double2 *__restrict__ vh_ie, double *partials, unsigned int *counter, DevScalars *sc) {
  __shared__ double2 s_d[SF2_ROWS][SF2_JT];
  __shared__ double s_red[32 + 1 + 1];
  const long long nrows = (long long)G.ny * G.nz;
  const long long row0 = (long long)blockIdx.x * SF2_ROWS;
  const int txb = blockDim.x;   // = (nx/2)/IXT
  double2 acc[IXT][SF2_ROWS];
#pragma unroll
  for (int q = 0; q < IXT; ++q)
#pragma unroll
    for (int r = 0; r < SF2_ROWS; ++r) acc[q][r] = make_double2(0.0, 0.0);
  for (int j0 = 0; j0 < nions; j0 += SF2_JT) {
    __syncthreads();
    for (int e = threadIdx.x; e < SF2_ROWS * SF2_JT; e += txb) {
      const int r = e / SF2_JT, jj = e % SF2_JT, j = j0 + jj;
      const long long row = row0 + r;
      double2 d = make_double2(0.0, 0.0);
      if (j < nions && row < nrows) {
        const int iy = (int)(row % G.ny), iz = (int)(row / G.ny);
        const double2 b = by_ij[(long long)iy * nions + j], c = cz_ij[(long long)iz * nions + j];
        const double z = Z[j];
        d = make_double2(z * (b.x * c.x - b.y * c.y), z * (b.x * c.y + b.y * c.x));
      }
      s_d[r][jj] = d;
    }
    __syncthreads();
    const int jn = min(SF2_JT, nions - j0);
    for (int jj = 0; jj < jn; ++jj) {
      double2 a[IXT];
#pragma unroll
      for (int q = 0; q < IXT; ++q) a[q] = ax_ji[(long long)(j0 + jj) * G.nx + threadIdx.x + q * txb];
#pragma unroll
      for (int r = 0; r < SF2_ROWS; ++r) {
        const double2 d = s_d[r][jj];
#pragma unroll
        for (int q = 0; q < IXT; ++q) {
          acc[q][r].x = fma(a[q].x, d.x, fma(-a[q].y, d.y, acc[q][r].x));
          acc[q][r].y = fma(a[q].x, d.y, fma(a[q].y, d.x, acc[q][r].y));
        }
      }
    }
  }
  double epm = 0.0;
#pragma unroll
  for (int q = 0; q < IXT; ++q) {
    const int ix = threadIdx.x + q * txb;
    const double wt = ix == 0 ? 1.0 : 2.0;
#pragma unroll
    for (int r = 0; r < SF2_ROWS; ++r) {
      const long long row = row0 + r;
      if (row < nrows) {
        const long long g = row * G.P + ix;
        S[g] = acc[q][r]; S2[g] = acc[q][r];
        const double v = vps[g];
        vh_ie[g] = make_double2(v * acc[q][r].x, v * acc[q][r].y);
        epm += wt * va[g] * (acc[q][r].x * acc[q][r].x + acc[q][r].y * acc[q][r].y);
      }
    }
  }
  double v[1] = {epm};
  const int op[1] = {0};
  if (grid_reduce<1>(v, op, partials, counter, s_red) && threadIdx.x == 0) sc->U_pm_sum = s_red[32];
}

// The same register tile fed by the copy engine (round 2).  ncu of the kernel above at 384^3 / 2000 ions: fp64 pipe 51%
// busy, long_scoreboard 4.3 warps per issue at the first DFMA that uses a_j(kx) -- the global loads of a_j are exposed,
// and a register prefetch only moves the stall (ptxas sinks the loads).  Here the a_j(kx) rows of
// SF3_JT ions at a time (one contiguous run of nx/2 complex numbers per ion) come into shared memory by cp.async.bulk
// completing on an mbarrier, two stages in flight, issued by one thread; d_j = Z_j b_j c_j of the next stage is fetched
// into registers before the current stage is consumed and written to the other half of a double buffer after it.  A
// block owns 8 RG rows (RG row groups share every a_j word).  Same outputs and the same closing reduction.
constexpr int SF3_JT = 8;
constexpr int SF3_NST = 2;
template <int IXT, int RG>
__global__ void __launch_bounds__(128, IXT * RG >= 12 ? 2 : 3) structure_factor_tma_kernel(
    GridGeom G, int nions, const double *__restrict__ Z, const double2 *__restrict__ ax_ji /*[j][ix]*/,
    const double2 *__restrict__ by_ij /*[iy][j]*/, const double2 *__restrict__ cz_ij /*[iz][j]*/,
    const double *__restrict__ vps, const double *__restrict__ va, double2 *__restrict__ S, double2 *__restrict__ S2,
    double2 *__restrict__ vh_ie, double *partials, unsigned int *counter, DevScalars *sc) {
  constexpr int ROWS = SF2_ROWS * RG, DE = ROWS * SF3_JT;   // rows per block; d_j elements per stage
  extern __shared__ __align__(16) double2 s_dyn[];
  __shared__ double s_red[32 + 1 + 1];
  __shared__ unsigned long long s_bar[SF3_NST];
  const int txb = blockDim.x / RG, nxm = IXT * txb;          // nxm = nx/2 columns
  double2 *s_a = s_dyn;                                      // [SF3_NST][SF3_JT][nxm]
  double2 *s_d = s_dyn + (size_t)SF3_NST * SF3_JT * nxm;     // [2][ROWS][SF3_JT]
  const int tid = threadIdx.x, tx = tid % txb, ty = tid / txb;
  const long long nrows = (long long)G.ny * G.nz, row0 = (long long)blockIdx.x * ROWS;
  const int nstages = (nions + SF3_JT - 1) / SF3_JT;
  for (int e = tid; e < SF3_NST * SF3_JT * nxm; e += blockDim.x) s_a[e] = make_double2(0.0, 0.0);
  fence_proxy_async();
  if (tid == 0)
    for (int q = 0; q < SF3_NST; ++q) mbar_init(&s_bar[q], 1);
  __syncthreads();
  auto issue = [&](int st) {   // thread 0: rows a_j(0 .. nx/2 - 1) of the ions of stage st
    const int q = st % SF3_NST, j0 = st * SF3_JT, nj = min(SF3_JT, nions - j0);
    mbar_arrive_expect_tx(&s_bar[q], (unsigned)(nj * nxm * sizeof(double2)));
    for (int jj = 0; jj < nj; ++jj)
      bulk_copy_g2s(s_a + ((size_t)q * SF3_JT + jj) * nxm, ax_ji + (long long)(j0 + jj) * G.nx, (unsigned)(nxm * sizeof(double2)), &s_bar[q]);
  };
  if (tid == 0)
    for (int st = 0; st < SF3_NST && st < nstages; ++st) issue(st);
  // the d_j elements this thread stages: element e = (row r, ion slot jj); its (iy, iz) never change
  constexpr int DPT = (DE + 127) / 128;
  int d_iy[DPT], d_iz[DPT];
  bool d_ok[DPT];
#pragma unroll
  for (int k = 0; k < DPT; ++k) {
    const int e = tid + k * 128, r = e / SF3_JT;
    const long long row = row0 + r;
    d_ok[k] = e < DE && row < nrows;
    d_iy[k] = d_ok[k] ? (int)(row % G.ny) : 0; d_iz[k] = d_ok[k] ? (int)(row / G.ny) : 0;
  }
  double2 fb[DPT], fc[DPT]; double fz[DPT];
  auto fetch = [&](int st) {
#pragma unroll
    for (int k = 0; k < DPT; ++k) {
      const int j = st * SF3_JT + (tid + k * 128) % SF3_JT;
      fz[k] = 0.0;
      if (d_ok[k] && j < nions) { fb[k] = by_ij[(long long)d_iy[k] * nions + j]; fc[k] = cz_ij[(long long)d_iz[k] * nions + j]; fz[k] = Z[j]; }
    }
  };
  auto stash = [&](int dbuf) {
#pragma unroll
    for (int k = 0; k < DPT; ++k) {
      const int e = tid + k * 128;
      if (e < DE) {
        double2 d = make_double2(0.0, 0.0);
        if (fz[k] != 0.0) d = make_double2(fz[k] * (fb[k].x * fc[k].x - fb[k].y * fc[k].y), fz[k] * (fb[k].x * fc[k].y + fb[k].y * fc[k].x));
        s_d[(size_t)dbuf * DE + e] = d;
      }
    }
  };
  double2 acc[IXT][SF2_ROWS];
#pragma unroll
  for (int q = 0; q < IXT; ++q)
#pragma unroll
    for (int r = 0; r < SF2_ROWS; ++r) acc[q][r] = make_double2(0.0, 0.0);
  fetch(0); stash(0);
  __syncthreads();
  for (int st = 0; st < nstages; ++st) {
    const int buf = st % SF3_NST, dbuf = st & 1;
    if (st + 1 < nstages) fetch(st + 1);
    mbar_wait(&s_bar[buf], (unsigned)((st / SF3_NST) & 1));
    const double2 *pa = s_a + (size_t)buf * SF3_JT * nxm + tx;
    const double2 *pd = s_d + (size_t)dbuf * DE + (size_t)ty * SF2_ROWS * SF3_JT;
#pragma unroll 2
    for (int jj = 0; jj < SF3_JT; ++jj) {
      double2 a[IXT];
#pragma unroll
      for (int q = 0; q < IXT; ++q) a[q] = pa[jj * nxm + q * txb];
#pragma unroll
      for (int r = 0; r < SF2_ROWS; ++r) {
        const double2 d = pd[r * SF3_JT + jj];
#pragma unroll
        for (int q = 0; q < IXT; ++q) {
          acc[q][r].x = fma(a[q].x, d.x, fma(-a[q].y, d.y, acc[q][r].x));
          acc[q][r].y = fma(a[q].x, d.y, fma(a[q].y, d.x, acc[q][r].y));
        }
      }
    }
    if (st + 1 < nstages) stash(dbuf ^ 1);
    __syncthreads();                                   // every warp is done with this stage's a_j rows and d_j
    if (tid == 0 && st + SF3_NST < nstages) issue(st + SF3_NST);
  }
  double epm = 0.0;
#pragma unroll
  for (int q = 0; q < IXT; ++q) {
    const int ix = tx + q * txb;
    const double wt = ix == 0 ? 1.0 : 2.0;
#pragma unroll
    for (int r = 0; r < SF2_ROWS; ++r) {
      const long long row = row0 + ty * SF2_ROWS + r;
      if (row < nrows) {
        const long long g = row * G.P + ix;
        S[g] = acc[q][r]; S2[g] = acc[q][r];
        const double v = vps[g];
        vh_ie[g] = make_double2(v * acc[q][r].x, v * acc[q][r].y);
        epm += wt * va[g] * (acc[q][r].x * acc[q][r].x + acc[q][r].y * acc[q][r].y);
      }
    }
  }
  double v[1] = {epm};
  const int op[1] = {0};
  if (grid_reduce<1>(v, op, partials, counter, s_red) && threadIdx.x == 0) sc->U_pm_sum = s_red[32];
}

// Nyquist planes (reading A6).  With the literal index set of P:142 a Nyquist component is +N/2, whose mirror -N/2 is
// not on the grid, so S_Z is not Hermitian there.  For every stored point with a Nyquist component this kernel forms
// S2 = S_Z(k''), k'' = k with every Nyquist component flipped to -N/2 (phase-table entries conjugated), and
//   Vhat_ie <- v(k) (S + S2)/2, the Hermitian part, whose half-spectrum inverse equals the real part of the full
//   inverse transform of v(k) S_Z(k);  sum conj(nhat) Vhat_ie over the half spectrum then equals Re sum over the full
//   literal set.  It also corrects the Ewald reciprocal energy for the mirrored halves of the y/z Nyquist rows.
// Points: list A = rows with ky or kz Nyquist (all stored kx), list B = the column kx = nx/2 of the other rows.
// One warp per point: the lanes stride over the ions (coalesced [k][j] tables), fixed-order shuffle reduction.
__global__ void __launch_bounds__(128) structure_factor_nyquist_kernel(
    GridGeom G, int nions, const double *__restrict__ Z, const double2 *__restrict__ ax_ij /*[ix][j]*/,
    const double2 *__restrict__ by_ij, const double2 *__restrict__ cz_ij, const double *__restrict__ vps,
    const double *__restrict__ va, double2 *S, double2 *__restrict__ S2, double2 *__restrict__ vh_ie,
    double *partials, unsigned int *counter, DevScalars *sc, int own_nyq_x /* 1: the main kernel left kx = nx/2 to this one */) {
  __shared__ double s_red[32 + 1 + 1];
  const int nyq_y = (G.ny % 2 == 0) ? G.ny / 2 : -1, nyq_z = (G.nz % 2 == 0) ? G.nz / 2 : -1;
  const int nyq_x = (G.nx % 2 == 0) ? G.nx / 2 : -1;
  const long long nrows = (long long)G.ny * G.nz;
  const int rowsA = (nyq_z >= 0 ? G.ny : 0) + (nyq_y >= 0 ? (nyq_z >= 0 ? G.nz - 1 : G.nz) : 0);
  const long long nA = (long long)rowsA * G.nxh, total = nA + (nyq_x >= 0 ? nrows : 0);
  const int lane = threadIdx.x & 31;
  const long long warp0 = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5, nwarps = ((long long)gridDim.x * blockDim.x) >> 5;
  double corr = 0.0;
  for (long long e = warp0; e < total; e += nwarps) {
    int ix, iy, iz;
    if (e < nA) {
      const int ra = (int)(e / G.nxh);
      ix = (int)(e % G.nxh);
      if (nyq_z >= 0 && ra < G.ny) { iy = ra; iz = nyq_z; }
      else { const int q = ra - (nyq_z >= 0 ? G.ny : 0); iy = nyq_y; iz = (nyq_z >= 0 && q >= nyq_z) ? q + 1 : q; }
    } else {
      const long long row = e - nA;
      ix = nyq_x; iy = (int)(row % G.ny); iz = (int)(row / G.ny);
      if (iy == nyq_y || iz == nyq_z) continue;   // already in list A
    }
    const bool fy = iy == nyq_y, fz = iz == nyq_z, fx = ix == nyq_x;
    const bool lit = own_nyq_x && fx;   // the literal S_Z of this point is computed here too
    double sr = 0.0, si = 0.0, lr = 0.0, li = 0.0;
    for (int j = lane; j < nions; j += 32) {
      double2 a = ax_ij[(long long)ix * nions + j], b = by_ij[(long long)iy * nions + j], c = cz_ij[(long long)iz * nions + j];
      const double z = Z[j];
      if (lit) {
        const double bcx = b.x * c.x - b.y * c.y, bcy = b.x * c.y + b.y * c.x;
        lr += z * (a.x * bcx - a.y * bcy); li += z * (a.x * bcy + a.y * bcx);
      }
      if (fx) a.y = -a.y;
      if (fy) b.y = -b.y;
      if (fz) c.y = -c.y;
      const double bcx = b.x * c.x - b.y * c.y, bcy = b.x * c.y + b.y * c.x;
      sr += z * (a.x * bcx - a.y * bcy); si += z * (a.x * bcy + a.y * bcx);
    }
    sr = warp_sum(sr); si = warp_sum(si);
    if (lit) { lr = warp_sum(lr); li = warp_sum(li); }
    if (lane == 0) {
      const long long g = ((long long)iz * G.ny + iy) * G.P + ix;
      if (lit) { S[g] = make_double2(lr, li); corr += va[g] * (lr * lr + li * li); }   // column weight 1 in Eq. 42
      const double2 s = S[g];
      S2[g] = make_double2(sr, si);
      const double v = vps[g];
      vh_ie[g] = make_double2(0.5 * v * (s.x + sr), 0.5 * v * (s.y + si));
      // interior columns were counted twice with |S|^2; the mirrored half carries |S2|^2 instead
      if (ix != 0 && !fx) corr += va[g] * ((sr * sr + si * si) - (s.x * s.x + s.y * s.y));
    }
  }
  double v[1] = {corr};
  const int op[1] = {0};
  if (grid_reduce<1>(v, op, partials, counter, s_red) && threadIdx.x == 0) sc->U_pm_fix = s_red[32];
}

// Ewald short-range part (Eq. 41, 46) with the minimum-image convention: one block per ion j.
__global__ void __launch_bounds__(128) ewald_pp_kernel(const double *__restrict__ pos, const double *__restrict__ Z,
                                                       int nions, double Lx, double Ly, double Lz, double alpha,
                                                       double *__restrict__ F_pp, double *__restrict__ e_pp) {
  __shared__ double s_red[4 * 32];
  const int j = blockIdx.x;
  const double xj = pos[3 * j], yj = pos[3 * j + 1], zj = pos[3 * j + 2], zq = Z[j];
  double fx = 0, fy = 0, fz = 0, en = 0;
  const double two_a_sqrtpi = 2.0 * alpha * 0.56418958354775628695;
  for (int k = threadIdx.x; k < nions; k += blockDim.x) {
    if (k == j) continue;
    double dx = xj - pos[3 * k], dy = yj - pos[3 * k + 1], dz = zj - pos[3 * k + 2];
    dx -= Lx * rint(dx / Lx); dy -= Ly * rint(dy / Ly); dz -= Lz * rint(dz / Lz);
    const double r2 = dx * dx + dy * dy + dz * dz, r = sqrt(r2);
    const double e = erfc(alpha * r) / r;
    const double q = zq * Z[k];
    en += 0.5 * q * e;
    const double fr = q * (e + two_a_sqrtpi * exp(-alpha * alpha * r2)) / r2;
    fx += fr * dx; fy += fr * dy; fz += fr * dz;
  }
  double v[4] = {fx, fy, fz, en};
  const int op[4] = {0, 0, 0, 0};
  block_reduce<4>(v, op, s_red);
  if (threadIdx.x == 0) { F_pp[3 * j] = v[0]; F_pp[3 * j + 1] = v[1]; F_pp[3 * j + 2] = v[2]; e_pp[j] = v[3]; }
}

// U_ii = U_pp + U_pm + U_je (Eq. 40-44); single block, fixed order.
__global__ void __launch_bounds__(256) ewald_finish_kernel(const double *__restrict__ e_pp, const double *__restrict__ Z,
                                                           int nions, double alpha, double vol, DevScalars *sc) {
  __shared__ double s_red[3 * 32];
  double a = 0, q = 0, q2 = 0;
  for (int j = threadIdx.x; j < nions; j += blockDim.x) { a += e_pp[j]; q += Z[j]; q2 += Z[j] * Z[j]; }
  double v[3] = {a, q, q2};
  const int op[3] = {0, 0, 0};
  block_reduce<3>(v, op, s_red);
  if (threadIdx.x == 0) {
    const double upm = 0.5 * (sc->U_pm_sum + sc->U_pm_fix) / vol - alpha * 0.56418958354775628695 * v[2];
    const double uje = -ARCHE_PI * v[1] * v[1] / (2.0 * alpha * alpha * vol);
    sc->U_pp = v[0];
    sc->U_ii = v[0] + upm + uje;
  }
}

// Forces.  F_j = -(2 pi/|Omega|) Z_j sum_k k Im( W(k) exp(-2 pi i k.r_j) ) over the literal index set of P:142,
//   W(k) = v(k) conj(nhat_a(k)) + V_alpha(k) conj(S_Z(k))   [electron-ion Eq. 56 + Ewald reciprocal Eq. 47],
// evaluated on the half spectrum: the term of a point and of its mirror are equal, so interior columns
// (0 < ix < nx/2) count twice and the self-mirrored columns ix = 0, nx/2 once.  On a row with a Nyquist ky or kz the
// mirror of (kx, +N/2, kz) is (-kx, -N/2, -kz), which the literal set replaces by (-kx, +N/2, -kz): such rows are
// summed as two variants, the literal one and (interior columns only) the one with the Nyquist component flipped
// (conjugated phase-table entry, S2 instead of S, -N/2 in the k factor).
// Block = FC_THREADS*IPT ions x one slab of (ky,kz) rows.  Register tile: every thread owns IPT ions and works on FC_RPT
// (virtual) rows at a time, so that one a_j(kx) load and one staged W(k) word feed FC_RPT resp. IPT complex products --
// with one ion and one row per thread the kernel is bound by its shared-memory/L1 reads (measured 0.35 of fp64 peak),
// not by the FMA pipe.  Per (ion, row, kx): t = W a_j, P += t, Q += kx t (8 fp64 instructions).
constexpr int FC_THREADS = 128;
constexpr int FC_RPT = 4;   // (virtual) rows in flight: every a_j(kx) word read from L2 feeds FC_RPT products
template <int IPT>
__global__ void __launch_bounds__(FC_THREADS) force_kernel(
    GridGeom G, int nions, int rows_per_slab, const double2 *__restrict__ ax_ij /*[ix][j]*/,
    const double2 *__restrict__ by_ij, const double2 *__restrict__ cz_ij, const double *__restrict__ vps,
    const double *__restrict__ va, const double2 *__restrict__ nh_a, const double2 *__restrict__ S,
    const double2 *__restrict__ S2, double *__restrict__ F_part /*[slab][j][3]*/) {
  extern __shared__ double2 s_w[];  // [FC_RPT][nxh] weighted W of the rows in flight, then kx[nxh]
  double *s_kx = reinterpret_cast<double *>(s_w + FC_RPT * G.nxh);
  const int j0 = blockIdx.x * (FC_THREADS * IPT) + threadIdx.x;
  const long long nrows = (long long)G.ny * G.nz;
  const long long r0 = (long long)blockIdx.y * rows_per_slab;
  const long long r1 = min(nrows, r0 + rows_per_slab);
  const int nyq_y = (G.ny % 2 == 0) ? G.ny / 2 : -1, nyq_z = (G.nz % 2 == 0) ? G.nz / 2 : -1;
  for (int ix = threadIdx.x; ix < G.nxh; ix += FC_THREADS) s_kx[ix] = G.kx[ix];
  double fx[IPT], fy[IPT], fz[IPT];
#pragma unroll
  for (int q = 0; q < IPT; ++q) fx[q] = fy[q] = fz[q] = 0.0;
  long long row = r0;
  int var = 0;
  while (row < r1) {
    // take up to FC_RPT virtual rows (row, variant)
    long long vrow[FC_RPT]; int vvar[FC_RPT]; bool vnyq[FC_RPT], vok[FC_RPT];
#pragma unroll
    for (int s = 0; s < FC_RPT; ++s) {
      vok[s] = row < r1; vrow[s] = vok[s] ? row : r0; vvar[s] = var;
      const int iy = (int)(vrow[s] % G.ny), iz = (int)(vrow[s] / G.ny);
      vnyq[s] = iy == nyq_y || iz == nyq_z;
      if (vok[s]) { if (vnyq[s] && var == 0) var = 1; else { ++row; var = 0; } }
    }
    __syncthreads();
#pragma unroll
    for (int s = 0; s < FC_RPT; ++s) {
      for (int ix = threadIdx.x; ix < G.nxh; ix += FC_THREADS) {
        double2 w = make_double2(0.0, 0.0);
        if (vok[s]) {
          const long long g = vrow[s] * G.P + ix;
          const bool edge = ix == 0 || 2 * ix == G.nx;
          const double wt = edge ? (vvar[s] == 0 ? 1.0 : 0.0) : (vnyq[s] ? 1.0 : 2.0);
          const double2 n = nh_a[g], sf = vvar[s] == 0 ? S[g] : S2[g];
          const double v = vps[g], a = va[g];
          w = make_double2(wt * (v * n.x + a * sf.x), -wt * (v * n.y + a * sf.y));
        }
        s_w[s * G.nxh + ix] = w;
      }
    }
    __syncthreads();
    double2 P[IPT][FC_RPT], Q[IPT][FC_RPT];
#pragma unroll
    for (int q = 0; q < IPT; ++q)
#pragma unroll
      for (int s = 0; s < FC_RPT; ++s) { P[q][s] = make_double2(0.0, 0.0); Q[q][s] = make_double2(0.0, 0.0); }
    for (int ix = 0; ix < G.nxh; ++ix) {
      double2 w[FC_RPT];
#pragma unroll
      for (int s = 0; s < FC_RPT; ++s) w[s] = s_w[s * G.nxh + ix];
      const double kx = s_kx[ix];
#pragma unroll
      for (int q = 0; q < IPT; ++q) {
        const int j = j0 + q * FC_THREADS;
        const double2 a = j < nions ? ax_ij[(long long)ix * nions + j] : make_double2(0.0, 0.0);
#pragma unroll
        for (int s = 0; s < FC_RPT; ++s) {
          const double2 t = make_double2(fma(w[s].x, a.x, -w[s].y * a.y), fma(w[s].x, a.y, w[s].y * a.x));
          P[q][s].x += t.x; P[q][s].y += t.y;
          Q[q][s].x = fma(kx, t.x, Q[q][s].x); Q[q][s].y = fma(kx, t.y, Q[q][s].y);
        }
      }
    }
#pragma unroll
    for (int s = 0; s < FC_RPT; ++s) {
      if (!vok[s]) continue;
      const int iy = (int)(vrow[s] % G.ny), iz = (int)(vrow[s] / G.ny);
#pragma unroll
      for (int q = 0; q < IPT; ++q) {
        const int j = j0 + q * FC_THREADS;
        if (j >= nions) continue;
        double2 b = by_ij[(long long)iy * nions + j], c = cz_ij[(long long)iz * nions + j];
        double ky = G.ky[iy], kz = G.kz[iz];
        if (vvar[s] == 1) {
          if (iy == nyq_y) { b.y = -b.y; ky = -ky; }
          if (iz == nyq_z) { c.y = -c.y; kz = -kz; }
        }
        const double2 bc = make_double2(b.x * c.x - b.y * c.y, b.x * c.y + b.y * c.x);
        const double imP = P[q][s].x * bc.y + P[q][s].y * bc.x, imQ = Q[q][s].x * bc.y + Q[q][s].y * bc.x;
        fx[q] += imQ; fy[q] += ky * imP; fz[q] += kz * imP;
      }
    }
  }
#pragma unroll
  for (int q = 0; q < IPT; ++q) {
    const int j = j0 + q * FC_THREADS;
    if (j < nions) {
      double *o = F_part + ((size_t)blockIdx.y * nions + j) * 3;
      o[0] = fx[q]; o[1] = fy[q]; o[2] = fz[q];
    }
  }
}

// Column-resident form of the force sum (round 2; n_ions >= 256).  ncu of force_kernel<4> at 384^3 / 2000 ions: 236
// registers, two blocks per SM, fp64 pipe 58% busy, the top stalls are the L2 loads of a_j(kx) (re-read for every group
// of four rows: 229 GB per call) and fixed-latency waits that two warps per scheduler cannot cover.  Here a thread
// owns one ion and CH kx columns and keeps a_j(kx) of those columns IN REGISTERS for its whole life; it walks over the
// (virtual) rows of its slab, and the only operand of the inner loop is W(row, kx), which the copy engine brings into
// shared memory (cp.async.bulk completing on an mbarrier, FCC_NST stages of FCC_GR rows in flight: no staging
// instructions in the compute warps) and every warp reads as a broadcast.  Per (ion, row, kx): t = W a_j, P += t,
// Q' += c t with the column number c an immediate (kx = (c0 + c)/Lx is linear in c: the kx-weighted sum is
// (c0 P + Q')/Lx), 8 fp64 instructions and one LDS.128; per (ion, row) 11 more to fold P, Q' with b_j(ky) c_j(kz) into
// the four running sums.
// Virtual rows: v < ny nz is row v in its literal form; v >= ny nz runs over the rows with a Nyquist ky or kz once more
// in the flipped variant (see force_kernel); the list is padded to a multiple of FCC_GR with rows of W = 0.
// force_rowinfo_kernel (once per context) tabulates iy, iz, the sign masks and the signed ky, kz of every virtual row;
// force_w_kernel (once per call) forms the weighted W of every virtual row: rows v < ny nz in Wa [ny nz][P] (the FFT
// scratch array), the others in Wb [.][P].  Grid of force_cols_kernel: x = tiles of 128 ions, y = column chunks, z =
// slabs of virtual rows; F_part[(z gridDim.y + y)][j][3].
constexpr int FCC_THREADS = 128;
constexpr int FCC_GR = 4;    // rows per shared-memory stage
constexpr int FCC_R = 2;     // rows in flight per thread
constexpr int FCC_NST = 3;   // stages in flight
struct ForceVRow { int iy, iz, var; bool nyq; };
__device__ __forceinline__ ForceVRow force_vrow(const GridGeom &G, int v, int nrows, int nyq_y, int nyq_z) {
  ForceVRow r;
  if (v < nrows) { r.iy = v % G.ny; r.iz = v / G.ny; r.var = 0; }
  else {
    const int ra = v - nrows;
    r.var = 1;
    if (nyq_z >= 0 && ra < G.ny) { r.iy = ra; r.iz = nyq_z; }
    else { const int q = ra - (nyq_z >= 0 ? G.ny : 0); r.iy = nyq_y; r.iz = (nyq_z >= 0 && q >= nyq_z) ? q + 1 : q; }
  }
  r.nyq = r.iy == nyq_y || r.iz == nyq_z;
  return r;
}
__host__ __device__ inline long long force_vrows(int ny, int nz) {   // virtual rows, not padded
  const bool ey = ny % 2 == 0, ez = nz % 2 == 0;
  return (long long)ny * nz + (ez ? ny : 0) + (ey ? (ez ? nz - 1 : nz) : 0);
}
__host__ __device__ inline long long force_vrows_padded(int ny, int nz) {
  return (force_vrows(ny, nz) + FCC_GR - 1) / FCC_GR * FCC_GR;
}
__device__ __forceinline__ double flip_sign(double x, unsigned int mask) {   // mask = 0 or 0x80000000
  return __hiloint2double(__double2hiint(x) ^ (int)mask, __double2loint(x));
}
__global__ void force_rowinfo_kernel(GridGeom G, int4 *__restrict__ ri, double2 *__restrict__ rk) {
  const int nrows = G.ny * G.nz, nv = (int)force_vrows(G.ny, G.nz), nvp = (int)force_vrows_padded(G.ny, G.nz);
  const int nyq_y = (G.ny % 2 == 0) ? G.ny / 2 : -1, nyq_z = (G.nz % 2 == 0) ? G.nz / 2 : -1;
  for (int v = blockIdx.x * blockDim.x + threadIdx.x; v < nvp; v += gridDim.x * blockDim.x) {
    if (v >= nv) { ri[v] = make_int4(0, 0, 0, 0); rk[v] = make_double2(0.0, 0.0); continue; }
    const ForceVRow r = force_vrow(G, v, nrows, nyq_y, nyq_z);
    const bool fy = r.var == 1 && r.iy == nyq_y, fz = r.var == 1 && r.iz == nyq_z;
    ri[v] = make_int4(r.iy, r.iz, fy ? (int)0x80000000u : 0, fz ? (int)0x80000000u : 0);
    rk[v] = make_double2(fy ? -G.ky[r.iy] : G.ky[r.iy], fz ? -G.kz[r.iz] : G.kz[r.iz]);
  }
}
__global__ void __launch_bounds__(256) force_w_kernel(GridGeom G, const double *__restrict__ vps, const double *__restrict__ va,
                                                      const double2 *__restrict__ nh_a, const double2 *__restrict__ S,
                                                      const double2 *__restrict__ S2, double2 *__restrict__ Wa,
                                                      double2 *__restrict__ Wb) {
  const int nrows = G.ny * G.nz, nv = (int)force_vrows(G.ny, G.nz), nvp = (int)force_vrows_padded(G.ny, G.nz);
  const int nyq_y = (G.ny % 2 == 0) ? G.ny / 2 : -1, nyq_z = (G.nz % 2 == 0) ? G.nz / 2 : -1;
  const long long tot = (long long)nvp * G.P;
  for (long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x; e < tot; e += (long long)gridDim.x * blockDim.x) {
    const int v = (int)(e / G.P), ix = (int)(e - (long long)v * G.P);
    double2 w = make_double2(0.0, 0.0);
    if (v < nv && ix < G.nxh) {
      const ForceVRow r = force_vrow(G, v, nrows, nyq_y, nyq_z);
      const long long g = ((long long)r.iz * G.ny + r.iy) * G.P + ix;
      const bool edge = ix == 0 || 2 * ix == G.nx;
      const double wt = edge ? (r.var == 0 ? 1.0 : 0.0) : (r.nyq ? 1.0 : 2.0);
      const double2 n = nh_a[g], sf = r.var == 0 ? S[g] : S2[g];
      const double pv = vps[g], pa = va[g];
      w = make_double2(wt * (pv * n.x + pa * sf.x), -wt * (pv * n.y + pa * sf.y));
    }
    if (v < nrows) Wa[e] = w; else Wb[e - (long long)nrows * G.P] = w;
  }
}
template <int CH>
__global__ void __launch_bounds__(FCC_THREADS, CH > 25 ? 2 : 3) force_cols_kernel(
    GridGeom G, int nions, int vrows_per_slab /* multiple of FCC_GR */, const double2 *__restrict__ ax_ij /*[ix][j]*/,
    const double2 *__restrict__ by_ij, const double2 *__restrict__ cz_ij, const double2 *__restrict__ Wa,
    const double2 *__restrict__ Wb, const int4 *__restrict__ ri_tab, const double2 *__restrict__ rk_tab,
    double *__restrict__ F_part) {
  static_assert(FCC_GR % FCC_R == 0, "rows in flight");
  __shared__ __align__(16) double2 s_w[FCC_NST][FCC_GR][CH];
  __shared__ __align__(16) int4 s_ri[FCC_NST][FCC_GR];      // iy, iz, sign masks of the flipped variant for b_j(ky).y, c_j(kz).y
  __shared__ __align__(16) double2 s_rk[FCC_NST][FCC_GR];   // ky, kz (signed for the flipped variant)
  __shared__ unsigned long long s_bar[FCC_NST];
  const int tid = threadIdx.x, j = blockIdx.x * FCC_THREADS + tid, c0 = blockIdx.y * CH;
  const bool jok = j < nions;
  const int jc = jok ? j : nions - 1;
  const int nrows = G.ny * G.nz, nvp = (int)force_vrows_padded(G.ny, G.nz);
  const int v0 = blockIdx.z * vrows_per_slab, v1 = min(nvp, v0 + vrows_per_slab);
  const int nstages = v1 > v0 ? (v1 - v0) / FCC_GR : 0;
  const int ncol = min(CH, G.P - c0);                        // columns of this chunk that exist in the arrays
  const unsigned stage_bytes = (unsigned)(FCC_GR * ncol * sizeof(double2) + FCC_GR * (sizeof(int4) + sizeof(double2)));
  for (int e = tid; e < FCC_NST * FCC_GR * CH; e += FCC_THREADS) (&s_w[0][0][0])[e] = make_double2(0.0, 0.0);
  fence_proxy_async();
  if (tid == 0)
    for (int q = 0; q < FCC_NST; ++q) mbar_init(&s_bar[q], 1);
  __syncthreads();
  auto issue = [&](int st) {   // thread 0: bring stage st into buffer st % FCC_NST
    const int q = st % FCC_NST, vb = v0 + st * FCC_GR;
    mbar_arrive_expect_tx(&s_bar[q], stage_bytes);
#pragma unroll
    for (int r = 0; r < FCC_GR; ++r) {
      const int v = vb + r;
      const double2 *src = v < nrows ? Wa + (long long)v * G.P + c0 : Wb + (long long)(v - nrows) * G.P + c0;
      bulk_copy_g2s(&s_w[q][r][0], src, (unsigned)(ncol * sizeof(double2)), &s_bar[q]);
    }
    bulk_copy_g2s(&s_ri[q][0], ri_tab + vb, FCC_GR * sizeof(int4), &s_bar[q]);
    bulk_copy_g2s(&s_rk[q][0], rk_tab + vb, FCC_GR * sizeof(double2), &s_bar[q]);
  };
  if (tid == 0)
    for (int st = 0; st < FCC_NST && st < nstages; ++st) issue(st);
  double2 a[CH];
#pragma unroll
  for (int c = 0; c < CH; ++c)
    a[c] = (jok && c0 + c < G.nxh) ? ax_ij[(long long)(c0 + c) * nions + j] : make_double2(0.0, 0.0);
  double sP = 0.0, sQ = 0.0, fy = 0.0, fz = 0.0;
  for (int st = 0; st < nstages; ++st) {
    const int buf = st % FCC_NST;
    mbar_wait(&s_bar[buf], (unsigned)((st / FCC_NST) & 1));
#pragma unroll
    for (int rr = 0; rr < FCC_GR; rr += FCC_R) {
      double2 b[FCC_R], cc[FCC_R];
#pragma unroll
      for (int q = 0; q < FCC_R; ++q) {
        const int4 ri = s_ri[buf][rr + q];
        b[q] = by_ij[(long long)ri.x * nions + jc]; cc[q] = cz_ij[(long long)ri.y * nions + jc];
        b[q].y = flip_sign(b[q].y, (unsigned int)ri.z); cc[q].y = flip_sign(cc[q].y, (unsigned int)ri.w);
      }
      double2 P[FCC_R], Q[FCC_R];
#pragma unroll
      for (int q = 0; q < FCC_R; ++q) { P[q] = make_double2(0.0, 0.0); Q[q] = make_double2(0.0, 0.0); }
#pragma unroll
      for (int c = 0; c < CH; ++c) {
#pragma unroll
        for (int q = 0; q < FCC_R; ++q) {
          const double2 w = s_w[buf][rr + q][c];
          const double2 t = make_double2(fma(w.x, a[c].x, -w.y * a[c].y), fma(w.x, a[c].y, w.y * a[c].x));
          P[q].x += t.x; P[q].y += t.y;
          if (c > 0) { Q[q].x = fma((double)c, t.x, Q[q].x); Q[q].y = fma((double)c, t.y, Q[q].y); }
        }
      }
#pragma unroll
      for (int q = 0; q < FCC_R; ++q) {
        const double2 k = s_rk[buf][rr + q];
        const double2 bc = make_double2(b[q].x * cc[q].x - b[q].y * cc[q].y, b[q].x * cc[q].y + b[q].y * cc[q].x);
        const double imP = P[q].x * bc.y + P[q].y * bc.x, imQ = Q[q].x * bc.y + Q[q].y * bc.x;
        sP += imP; sQ += imQ; fy = fma(k.x, imP, fy); fz = fma(k.y, imP, fz);
      }
    }
    __syncthreads();                                   // every warp is done with this buffer
    if (tid == 0 && st + FCC_NST < nstages) issue(st + FCC_NST);
  }
  if (jok) {
    double *o = F_part + ((size_t)(blockIdx.z * gridDim.y + blockIdx.y) * nions + j) * 3;
    o[0] = ((double)c0 * sP + sQ) / G.Lx; o[1] = fy; o[2] = fz;
  }
}

// one warp per force component: the lanes stride over the slabs, fixed-order shuffle tree (deterministic)
__global__ void force_finish_kernel(int nions, int nslabs, const double *__restrict__ F_part, const double *__restrict__ F_pp,
                                    const double *__restrict__ Z, double pref /* -2 pi/|Omega| */, double *__restrict__ F) {
  const int e = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
  if (e >= 3 * nions) return;
  double a = 0.0;
  for (int s = lane; s < nslabs; s += 32) a += F_part[(size_t)s * nions * 3 + e];
  a = warp_sum(a);
  if (lane == 0) F[e] = pref * Z[e / 3] * a + F_pp[e];
}

// velocity Verlet pieces (reading D2)
__global__ void kick_drift_kernel(double *__restrict__ pos, double *__restrict__ vel, const double *__restrict__ F,
                                  const double *__restrict__ mass, double dt, int nions, int drift) {
  const int e = blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= 3 * nions) return;
  const double v = vel[e] + 0.5 * dt * F[e] / mass[e / 3];
  vel[e] = v;
  if (drift) pos[e] += dt * v;
}

// Isokinetic ensemble (ref. [48]; reading A23): the exact flow over a time t of the Gaussian isokinetic
// equations m dv/dt = F - alpha m v, alpha = sum F.v / sum m v^2, with the forces held constant, followed (drift = 1) by
// the position update.  v(t) = (v(0) + (F/m) s)/s', s'' = a + b s with a = sum F.v/(2K), b = sum F^2/m /(2K); expm1 keeps
// cosh - 1 exact for the small arguments of an MD step.  One block: the three sums are O(N_i).
__global__ void __launch_bounds__(1024) isokinetic_kick_kernel(double *__restrict__ pos, double *__restrict__ vel,
                                                               const double *__restrict__ F, const double *__restrict__ mass,
                                                               double t, double dt, int nions, int drift) {
  __shared__ double s_red[3 * 32];
  __shared__ double s_s, s_sd;
  double v[3] = {0.0, 0.0, 0.0};
  for (int e = threadIdx.x; e < 3 * nions; e += blockDim.x) {
    const double m = mass[e / 3], u = vel[e], f = F[e];
    v[0] = fma(m * u, u, v[0]); v[1] = fma(f, u, v[1]); v[2] = fma(f / m, f, v[2]);
  }
  const int op[3] = {0, 0, 0};
  block_reduce<3>(v, op, s_red);
  if (threadIdx.x == 0) {
    double s = 0.0, sd = 1.0;   // no motion to constrain, or no force: v stays
    if (v[0] > 0.0 && v[2] > 0.0) {
      const double a = v[1] / v[0], b = v[2] / v[0], rb = sqrt(b), x = t * rb;
      const double ep = expm1(x), em = expm1(-x), sh = 0.5 * (ep - em), chm1 = 0.5 * (ep + em);
      s = (a / b) * chm1 + sh / rb;
      sd = (a / rb) * sh + chm1 + 1.0;
    }
    s_s = s; s_sd = sd;
  }
  __syncthreads();
  const double s = s_s, rsd = 1.0 / s_sd;
  for (int e = threadIdx.x; e < 3 * nions; e += blockDim.x) {
    const double u = (vel[e] + F[e] / mass[e / 3] * s) * rsd;
    vel[e] = u;
    if (drift) pos[e] += dt * u;
  }
}

__global__ void __launch_bounds__(256) kinetic_kernel(const double *__restrict__ vel, const double *__restrict__ mass,
                                                      int nions, DevScalars *sc) {
  __shared__ double s_red[32];
  double a = 0.0;
  for (int e = threadIdx.x; e < 3 * nions; e += blockDim.x) a += 0.5 * mass[e / 3] * vel[e] * vel[e];  // Eq. 36
  double v[1] = {a};
  const int op[1] = {0};
  block_reduce<1>(v, op, s_red);
  if (threadIdx.x == 0) sc->K_i = v[0];
}

}  // namespace arche
