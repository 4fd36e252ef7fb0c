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
};

template <int NX, int NY, int NZ>
constexpr size_t persist_smem_bytes() {
  constexpr size_t gy = 256 / fast_threads_yz<NY>(), gz = 256 / fast_threads_yz<NZ>();
  constexpr size_t ty = gy * NY * kFastL * sizeof(double2), tz = gz * NZ * kFastL * sizeof(double2);
  constexpr size_t tx = (size_t)kFastLP * fast_row_x<NX>() * sizeof(double2);
  constexpr size_t tile = ty > tz ? (ty > tx ? ty : tx) : (tz > tx ? tz : tx);
  return (kFdTabDoubles + kMaxRed * 33 + 8) * sizeof(double) + tile;
}

template <int N, int AXIS, bool INVERSE, class LoadOp, class StoreOp>
__device__ __forceinline__ void persist_yz_phase(const FastGeom &G, LoadOp &ld, StoreOp &st, double2 *tiles, int ntiles) {
  constexpr int TH = fast_threads_yz<N>(), GR = 256 / TH;
  const int group = threadIdx.x / TH, t = threadIdx.x % TH;
  for (int tile = blockIdx.x + gridDim.x * group; tile < ntiles; tile += gridDim.x * GR)
    fft_yz_tile<N, AXIS, INVERSE, false>(G, ld, st, tile, tiles + (size_t)group * N * kFastL, t, 1 + group);
}

template <int NX, int NY, int NZ>
__global__ void __launch_bounds__(256, 1) scf_persistent_kernel(PersistParams p) {
  namespace cg = cooperative_groups;
  cg::grid_group grid = cg::this_grid();
  extern __shared__ double smem[];
  double *s_tab = smem;
  double *s_red = s_tab + kFdTabDoubles;
  double *s_bc = s_red + kMaxRed * 33;
  double2 *tiles = reinterpret_cast<double2 *>(s_bc + 8);
  fd_load_tables(s_tab, p.fdtab);
  __syncthreads();
  const FastGeom Gx{NX, NY, NZ, p.P, p.tw0, nullptr}, Gy{NX, NY, NZ, p.P, p.tw1, nullptr}, Gz{NX, NY, NZ, p.P, p.tw2, nullptr};
  const int xtiles = NY * NZ / (2 * kFastLP), ytiles = NZ * (p.P / kFastL), ztiles = NY * (p.P / kFastL);
  int mix = p.mix_first;
  for (int it = 0; it < p.max_iters; ++it) {
    // ---- S1 (+ pending S6 in G-space): inverse z pass
    {
      LoadPotentialG lp;
      lp.nh_i = p.nh_i; lp.nh_a = p.nh_a; lp.vh_ie = p.vh_ie; lp.kx2 = p.kx2; lp.ky2 = p.ky2; lp.kz2 = p.kz2;
      lp.sc = p.sc; lp.nxh = p.nxh; lp.mix = mix;
      StoreComplex sw{p.work};
      lp.begin();
      persist_yz_phase<NZ, 2, true>(Gz, lp, sw, tiles, ztiles);
    }
    grid.sync();
    {
      LoadComplex lw{p.work};
      StoreComplex sw{p.work};
      persist_yz_phase<NY, 1, true>(Gy, lw, sw, tiles, ytiles);
    }
    grid.sync();
    // ---- S2 (+ pending S6 in real space, + first mu evaluation): c2r x pass
    {
      LoadComplex lw{p.work};
      StoreVi sv;
      sv.V_i = p.V_i; sv.n_i = p.n_i; sv.n_a = p.n_a; sv.sc = p.sc; sv.partials = p.partials; sv.counter = p.counter;
      sv.fdtab = s_tab; sv.inv_vol = p.inv_vol; sv.kT_eta0 = p.C.kT * p.C.eta0; sv.inv_kT = 1.0 / p.C.kT; sv.xc = p.C.xc;
      sv.mix = mix;
      sv.begin();
      for (int tile = blockIdx.x; tile < xtiles; tile += gridDim.x) fft_c2r_tile<NX, false>(Gx, lw, sv, tile, tiles);
      sv.finish(s_red);
    }
    grid.sync();
    // ---- S3: mu (grid barriers inside, one per evaluation)
    const double mu = mu_solve_dev(grid, p.V_i, p.ng, p.C, p.sc, s_tab, s_red, s_bc,
                                   p.partials + (size_t)gridDim.x * kMaxRed, p.mu_max_pass);
    // ---- S4: density prologue of the r2c x pass
    {
      LoadDensity ldn;
      ldn.V_i = p.V_i; ldn.n_i = p.n_i; ldn.n_a = p.n_a; ldn.sc = p.sc; ldn.partials = p.partials; ldn.counter = p.counter;
      ldn.fdtab = s_tab; ldn.C = p.C;
      StoreComplex sw{p.work};
      ldn.begin();
      ldn.mu = mu;   // block 0's store to sc->mu may not be visible yet; every block holds the same value
      for (int tile = blockIdx.x; tile < xtiles; tile += gridDim.x) fft_r2c_tile<NX, false>(Gx, ldn, sw, tile, tiles);
      ldn.finish(s_red);
    }
    grid.sync();
    {
      LoadComplex lw{p.work};
      StoreComplex sw{p.work};
      persist_yz_phase<NY, 1, false>(Gy, lw, sw, tiles, ytiles);
    }
    grid.sync();
    // ---- S5 (+ w, F, stop flag): forward z pass
    {
      LoadComplex lw{p.work};
      StoreNhatA sn;
      sn.nh_a = p.nh_a; sn.nh_i = p.nh_i; sn.vh_ie = p.vh_ie; sn.kx2 = p.kx2; sn.ky2 = p.ky2; sn.kz2 = p.kz2;
      sn.sc = p.sc; sn.partials = p.partials; sn.counter = p.counter; sn.C = p.C; sn.H.nx = NX; sn.H.nxh = p.nxh;
      sn.prestored = 0;
      sn.begin();
      persist_yz_phase<NZ, 2, false>(Gz, lw, sn, tiles, ztiles);
      __syncthreads();
      sn.finish(s_red);
    }
    grid.sync();
    mix = 1;
    if (!p.fixed && __ldcg(&p.sc->converged)) break;
  }
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
  return cudaLaunchCooperativeKernel(kern, dim3(blocks), dim3(256), args, smem, stream);
}

}  // namespace arche
