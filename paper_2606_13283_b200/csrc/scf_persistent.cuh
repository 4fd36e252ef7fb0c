// scf_persistent.cuh -- the whole SCF solve (S1..S7) of an L2-resident grid in ONE cooperative launch.
//
// On 32^3 / 64^3 grids every pass of the per-pass form lasts 4-17 us, most of it launch ramp, dependent latency chains
// and the drain of a 256-320 block grid; an SCF iteration is 7 such launches and a solve is ~160 iterations.  Here one
// block per SM stays resident for the whole solve: the same tile functions (fft_fast.cuh) and the same functors
// (scf_kernels.cuh) run phase by phase, separated by grid-wide barriers; the Fermi-Dirac table is loaded into shared
// memory once; the host reads the scalar block once per solve.  Results are those of the per-pass form up to the
// order of the deterministic partial sums (the partial-sum layout follows the grid size).
//
// Work distribution per phase: y/z passes -- groups of fast_threads_yz<N>() threads (4 groups per block at N = 64), one
// tile per group and round, named barriers per group; x passes -- the whole block per tile.
#pragma once
#include <cooperative_groups.h>

#include "fft_fast.cuh"
#include "scf_kernels.cuh"

namespace arche {

struct PersistParams {
  double *n_i, *n_a, *V_i;
  double2 *nh_i, *nh_a, *work;
  const double2 *vh_ie;
  const double *kx2, *ky2, *kz2;
  const double2 *tw0, *tw1, *tw2;
  DevScalars *sc;
  double *partials;
  unsigned int *counter;
  const double *fdtab;
  ScfConst C;
  int nxh, P;
  long long ng;
  double inv_vol;
  int mix_first;   // a mixing step of an earlier iteration is still pending when the solve starts
  int max_iters;   // iterations to run at most (exactly, when fixed)
  int fixed;       // 1: ignore the stop flag (parity replay)
  int mu_max_pass;
  unsigned long long *phase_ns;   // optional [8]: nanoseconds per phase (7 phases incl. their barrier) + iteration count
};

constexpr int kPersistThreads = 256;     // measured on c2: 512 threads (one pair element per thread and x tile) is slower
constexpr int kPersistBlocksPerSM = 1;   // measured on c2: 2 blocks/SM shortens the x phases but lengthens the barriers

template <int NX, int NY, int NZ>
constexpr size_t persist_smem_bytes() {
  constexpr size_t gy = kPersistThreads / fast_threads_yz<NY>(), gz = kPersistThreads / fast_threads_yz<NZ>();
  constexpr size_t ty = gy * NY * kFastL * sizeof(double2), tz = gz * NZ * kFastL * sizeof(double2);
  constexpr size_t tx = 2 * (size_t)kFastLP * fast_row_x<NX>() * sizeof(double2);   // two x tiles at a time
  constexpr size_t tile = ty > tz ? (ty > tx ? ty : tx) : (tz > tx ? tz : tx);
  return (kFdTabDoubles + 10 * 33 + 8 + 2 * (NX + NY + NZ) + (NX + NY + NZ)) * sizeof(double) + tile;
}

template <int N, int AXIS, bool INVERSE, class LoadOp, class StoreOp>
__device__ __forceinline__ void persist_yz_phase(const FastGeom &G, LoadOp &ld, StoreOp &st, double2 *tiles, int ntiles) {
  constexpr int TH = fast_threads_yz<N>(), GR = kPersistThreads / TH;
  const int group = threadIdx.x / TH, t = threadIdx.x % TH;
  for (int tile = blockIdx.x + gridDim.x * group; tile < ntiles; tile += gridDim.x * GR)
    fft_yz_tile<N, AXIS, INVERSE, false>(G, ld, st, tile, tiles + (size_t)group * N * kFastL, t, 1 + group);
}

template <int NX, int NY, int NZ>
__global__ void __launch_bounds__(kPersistThreads, kPersistBlocksPerSM) scf_persistent_kernel(PersistParams p) {
  namespace cg = cooperative_groups;
  cg::grid_group grid = cg::this_grid();
  extern __shared__ __align__(16) double smem[];
  double *s_tab = smem;
  double *s_red = s_tab + kFdTabDoubles;
  double *s_bc = s_red + 10 * 33;
  double2 *s_tw0 = reinterpret_cast<double2 *>(s_bc + 8), *s_tw1 = s_tw0 + NX, *s_tw2 = s_tw1 + NY;   // twiddles
  double *s_kx2 = reinterpret_cast<double *>(s_tw2 + NZ), *s_ky2 = s_kx2 + NX, *s_kz2 = s_ky2 + NY;    // k^2 per axis
  double2 *tiles = reinterpret_cast<double2 *>(s_kz2 + NZ);
  for (int i = threadIdx.x; i < NX; i += blockDim.x) { s_tw0[i] = p.tw0[i]; s_kx2[i] = p.kx2[i]; }
  for (int i = threadIdx.x; i < NY; i += blockDim.x) { s_tw1[i] = p.tw1[i]; s_ky2[i] = p.ky2[i]; }
  for (int i = threadIdx.x; i < NZ; i += blockDim.x) { s_tw2[i] = p.tw2[i]; s_kz2[i] = p.kz2[i]; }
  // every block keeps its own copy of the scalar block in shared memory: the phase totals are taken by all blocks
  // in the same fixed order after a grid barrier (block_partials / block_totals), so the copies stay identical and no
  // block ever waits for another one's scalar result; block 0 writes the copy back at the end
  __shared__ DevScalars s_sc;
  if (threadIdx.x == 0) s_sc = *p.sc;
  __shared__ unsigned long long s_bar;
  fd_load_tables(s_tab, p.fdtab, &s_bar);
  __syncthreads();
  DevScalars *const sc = &s_sc;
  double *const part_vi = p.partials, *const part_dg = part_vi + (size_t)gridDim.x * 4,   // density 7 + G-space 3 per block
         *const part_mu = part_dg + (size_t)gridDim.x * 10;
  const FastGeom Gx{NX, NY, NZ, p.P, s_tw0, nullptr}, Gy{NX, NY, NZ, p.P, s_tw1, nullptr}, Gz{NX, NY, NZ, p.P, s_tw2, nullptr};
  constexpr int XTH = kPersistThreads / 2;   // two x tiles per block at a time
  const int xg = threadIdx.x / XTH, xt = threadIdx.x % XTH;
  double2 *const xbuf = tiles + (size_t)xg * kFastLP * fast_row_x<NX>();
  const int xtiles = NY * NZ / (2 * kFastLP), ytiles = NZ * (p.P / kFastL), ztiles = NY * (p.P / kFastL);
  int mix = p.mix_first;
  const bool timing = p.phase_ns != nullptr && blockIdx.x == 0 && threadIdx.x == 0;
  unsigned long long t_prev = 0;
  auto lap = [&](int phase) {   // block 0 attributes the time since the previous lap (work + barrier) to `phase`
    if (timing) {
      unsigned long long t;
      asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
      if (phase >= 0) p.phase_ns[phase] += t - t_prev;
      t_prev = t;
    }
  };
  lap(-1);
  for (int it = 0; it < p.max_iters; ++it) {
    // ---- S1 (+ pending S6 in G-space): inverse z pass
    {
      LoadPotentialG lp;
      lp.nh_i = p.nh_i; lp.nh_a = p.nh_a; lp.vh_ie = p.vh_ie; lp.kx2 = s_kx2; lp.ky2 = s_ky2; lp.kz2 = s_kz2;
      lp.sc = sc; lp.nxh = p.nxh; lp.mix = mix;
      StoreComplex sw{p.work};
      lp.begin();
      persist_yz_phase<NZ, 2, true>(Gz, lp, sw, tiles, ztiles);
    }
    grid.sync();
    lap(0);
    {
      LoadComplex lw{p.work};
      StoreComplex sw{p.work};
      persist_yz_phase<NY, 1, true>(Gy, lw, sw, tiles, ytiles);
    }
    grid.sync();
    lap(1);
    // ---- S2 (+ pending S6 in real space, + first mu evaluation): c2r x pass
    {
      LoadComplex lw{p.work};
      StoreVi sv;
      sv.V_i = p.V_i; sv.n_i = p.n_i; sv.n_a = p.n_a; sv.sc = sc; sv.partials = nullptr; sv.counter = nullptr;
      sv.fdtab = s_tab; sv.inv_vol = p.inv_vol; sv.kT_eta0 = p.C.kT * p.C.eta0; sv.inv_kT = 1.0 / p.C.kT; sv.xc = p.C.xc;
      sv.mix = mix;
      sv.begin();
      for (int tile = blockIdx.x + gridDim.x * xg; tile < xtiles; tile += 2 * gridDim.x)
        fft_c2r_tile<NX, false, XTH>(Gx, lw, sv, tile, xbuf, xt, 1 + xg);
      __syncthreads();
      sv.partial(s_red, part_vi);
    }
    grid.sync();
    {
      double t[4];
      const int op[4] = {1, 2, 0, 0};
      block_totals<4>(op, part_vi, s_red, t);
      if (threadIdx.x == 0) StoreVi::apply(t, p.C.kT * p.C.eta0, sc);
      __syncthreads();
    }
    lap(2);
    // ---- S3: mu (grid barriers inside, one per evaluation)
    const double mu = mu_solve_dev(grid, p.V_i, p.ng, p.C, sc, s_tab, s_red, s_bc, part_mu, p.mu_max_pass, true);
    __syncthreads();
    lap(3);
    // ---- S4: density prologue of the r2c x pass
    {
      LoadDensity ldn;
      ldn.V_i = p.V_i; ldn.n_i = p.n_i; ldn.n_a = p.n_a; ldn.sc = sc; ldn.partials = nullptr; ldn.counter = nullptr;
      ldn.fdtab = s_tab; ldn.C = p.C;
      StoreComplex sw{p.work};
      ldn.begin();
      ldn.mu = mu;
      for (int tile = blockIdx.x + gridDim.x * xg; tile < xtiles; tile += 2 * gridDim.x)
        fft_r2c_tile<NX, false, XTH>(Gx, ldn, sw, tile, xbuf, xt, 1 + xg);
      __syncthreads();
      ldn.partial(s_red, part_dg, 10, 0);
    }
    grid.sync();
    lap(4);
    {
      LoadComplex lw{p.work};
      StoreComplex sw{p.work};
      persist_yz_phase<NY, 1, false>(Gy, lw, sw, tiles, ytiles);
    }
    grid.sync();
    lap(5);
    // ---- S5 (+ w, F, stop flag): forward z pass
    {
      LoadComplex lw{p.work};
      StoreNhatA sn;
      sn.nh_a = p.nh_a; sn.nh_i = p.nh_i; sn.vh_ie = p.vh_ie; sn.kx2 = s_kx2; sn.ky2 = s_ky2; sn.kz2 = s_kz2;
      sn.sc = sc; sn.partials = nullptr; sn.counter = nullptr; sn.C = p.C; sn.H.nx = NX; sn.H.nxh = p.nxh;
      sn.prestored = 0;
      sn.begin();
      persist_yz_phase<NZ, 2, false>(Gz, lw, sn, tiles, ztiles);
      __syncthreads();
      sn.partial(s_red, part_dg, 10, 7);
    }
    grid.sync();
    {  // totals of the density pass and of the G-space pass -> K, F0, ..., then U, E_H, E_ie, w, F and the stop flag
      double t[10];
      const int op[10] = {0, 0, 0, 0, 0, 0, 0, 0, 0, 0};
      block_totals<10>(op, part_dg, s_red, t);
      if (threadIdx.x == 0) { LoadDensity::apply(t, p.C, sc); StoreNhatA::apply(t + 7, p.C, sc); }
      __syncthreads();
    }
    lap(6);
    if (timing) p.phase_ns[7] += 1;
    mix = 1;
    if (!p.fixed && sc->converged) break;
  }
  if (blockIdx.x == 0 && threadIdx.x == 0) *p.sc = s_sc;
}

// launches the persistent solve when the grid has an instantiation; cudaErrorNotSupported otherwise
static inline cudaError_t scf_persistent_launch(int nx, int ny, int nz, const PersistParams &p, int blocks, cudaStream_t stream) {
  const void *kern = nullptr;
  size_t smem = 0;
  if (nx == 32 && ny == 32 && nz == 32) { kern = (const void *)scf_persistent_kernel<32, 32, 32>; smem = persist_smem_bytes<32, 32, 32>(); }
  else if (nx == 64 && ny == 64 && nz == 64) { kern = (const void *)scf_persistent_kernel<64, 64, 64>; smem = persist_smem_bytes<64, 64, 64>(); }
  else return cudaErrorNotSupported;
  cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return e;
  PersistParams pp = p;
  void *args[] = {&pp};
  return cudaLaunchCooperativeKernel(kern, dim3(blocks), dim3(kPersistThreads), args, smem, stream);
}

}  // namespace arche
