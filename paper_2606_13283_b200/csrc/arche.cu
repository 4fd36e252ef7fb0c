// arche.cu -- host control + C ABI (include/arche.h) of the B200 Thomas-Fermi SCF / OFMD hot path.
// Every step of the path runs in the CUDA kernels of fft.cuh, scf_kernels.cuh and ion_kernels.cuh; the host only
// sequences launches on the caller's stream and reads one small scalar block per SCF iteration.
#include "../../include/arche.h"

#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <new>
#include <vector>

#include "common.cuh"
#include "fd.cuh"
#include "fft.cuh"
#include "fft_fast.cuh"
#include "ion_kernels.cuh"
#include "scf_kernels.cuh"
#include "scf_persistent.cuh"
#include "stress_kernels.cuh"
#include "peak_kernels.cuh"

using namespace arche;

namespace {

constexpr int kMuMaxPasses = 12;
constexpr int kScfBatch = 6;      // SCF iterations launched between two reads of the device scalars
constexpr int kProfPairs = 512;
// kernel classes for arche_profile_get
enum ProfClass { PC_FFT_INV_Z = 0, PC_FFT_Y, PC_FFT_INV_X, PC_MU, PC_DENSITY, PC_FFT_FWD_X, PC_FFT_FWD_Z, PC_MIX,
                 PC_SFAC, PC_FORCE, PC_EWALD, PC_OTHER, PC_POT_G, PC_VI_R, PC_DENS_R, PC_RED_G, PC_STRESS, kProfClasses };
constexpr int kEwBlocks = 148 * 8;

inline size_t align256(size_t x) { return (x + 255) & ~(size_t)255; }

struct Carver {  // carves 256-byte aligned arrays out of the caller's workspace (or just measures)
  char *base;
  size_t off;
  template <class T> T *take(size_t count) {
    T *p = base ? reinterpret_cast<T *>(base + off) : nullptr;
    off += align256(count * sizeof(T));
    return p;
  }
};

// host evaluation of the same fits (only for eta0 = I_{1/2}^{-1}(Ne/(|Omega| cTF)), once per init)
double fd_host(int f, double eta) {  // f = 0, 1, 2: I_{-1/2}, I_{1/2}, I_{3/2}
  int seg; double t, p[3];
  fd_locate(eta, seg, t, p[0], p[1], p[2]);
  double a = FD_COEF[f][seg][FD_NC - 1];
  for (int i = FD_NC - 2; i >= 0; --i) a = fma(a, t, FD_COEF[f][seg][i]);
  return a * p[f];
}
double fd_half_host(double eta) { return fd_host(1, eta); }
double fd_half_inverse_host(double y) {
  double lo = log(y / 0.88622692545275801365), hi = pow(1.5 * y, 2.0 / 3.0) + 2.0;
  if (hi < lo + 2.0) hi = lo + 2.0;
  for (int it = 0; it < 200; ++it) {
    double mid = 0.5 * (lo + hi);
    if (mid == lo || mid == hi) break;
    if (fd_half_host(mid) < y) lo = mid; else hi = mid;
  }
  return 0.5 * (lo + hi);
}

bool grid_ok(int n) {
  if (n < 4 || n > 1024) return false;
  while (n % 2 == 0) n /= 2;
  while (n % 3 == 0) n /= 3;
  return n == 1;
}

}  // namespace

struct arche_ctx {
  arche_params p;
  cudaStream_t stream;
  GridGeom G;
  ScfConst C;
  long long ng;
  int nions;
  double alpha, Q;
  FftAxisPlan plan[3];
  int red_blocks;  // capacity of the partials buffer (blocks)
  int mu_grid;     // co-resident blocks of the cooperative mu/density kernel
  int ew_grid;     // blocks of grid-stride elementwise kernels
  bool mu_regular; int mu_coop_iters;   // mu as ordinary launches only from iteration mu_coop_iters of a solve (ARCHE_MU_REGULAR, ARCHE_MU_COOP_ITERS)
  bool mu_split;   // first evaluation of the mu iteration as an ordinary launch (mu_first_eval_kernel; ARCHE_MU_SPLIT=0: off)
  bool r2c_tma;    // plain r2c x pass fed by the copy engine (ARCHE_R2C_TMA)
  bool sf_tma;     // structure factor: register tile fed by the copy engine (ARCHE_SF_TMA=0: global loads of a_j)
  bool s5_rows;    // S5 reduction of the streamed form as a row walk (ARCHE_S5_ROWS=0: the generic grid-stride kernel)
  bool lazy_F;     // free energy only where the stop rule needs it (ARCHE_LAZY_F=0 disables); see ScfConst::lazy_F
  bool pdl;        // programmatic dependent launch between the kernels of an SCF iteration (ARCHE_PDL=0 disables)
  int r_blocks;    // resident blocks per SM of the streamed real-space Fermi-Dirac kernels
  int force_slabs, force_rows_per_slab, force_ipt;   // ions per thread of the force kernel's register tile
  int force_ch, force_chunks, force_zslabs;          // > 0: column-resident force kernel with force_ch columns per thread
  double2 *force_wb, *force_rk;                      // W of the flipped Nyquist rows; signed ky, kz per virtual row
  int4 *force_ri;                                    // iy, iz, sign masks per virtual row
  // device arrays (all inside the caller's workspace)
  double *n_i, *n_a, *V_i, *vps, *va, *psp_tab;
  PspTable T;      // f2: tabulated pseudopotential (device table inside the workspace)
  double2 *nh_i, *nh_a, *vh_ie, *S, *S2, *gh, *gh2, *work;  // half spectrum [nz][ny][P]
  double2 *fft_static = nullptr;   // device address of g_fft3d_static_scratch on this context's device
  long long nh;      // P*ny*nz
  int nxh, P;
  bool persist;      // whole solve in one cooperative launch (scf_persistent.cuh): fused form, 32^3 / 64^3 grids
  int sm_count;
  const int *stop;   // device flag handed to the kernels of speculatively launched iterations (nullptr: never skip)
  bool fuse;         // pointwise work fused into the FFT passes (grids that live in L2) or streamed around plain passes
  bool use_fast;     // register two-stage FFT passes where the axis length has a plan (ARCHE_FFT_GENERIC=1 disables)
  bool mix_pending;  // S6 of the last iteration not yet applied to n_i / nhat_i (fused into the next S1/S2)
  double *kx, *ky, *kz, *kx2, *ky2, *kz2;
  double2 *tw[3];
  double2 *ax_ij, *ax_ji, *by_ij, *cz_ij;
  double *Z, *mass, *pos, *F, *F_pp, *e_pp, *F_part, *vel_tmp;
  double *pp_part, *stress;   // [nions][6] short-range stress sums; [64] assembled table (device)
  double *h_stress;           // pinned [64]
  double *fdtab, *partials;
  unsigned int *counter;
  unsigned long long *phase_ns;
  DevScalars *sc;
  DevScalars *h_sc;  // pinned
  bool have_g, have_solution, have_forces;
  long long launches;
  // optional per-kernel-class timing (CUDA events on c->stream), see arche_profile_*
  bool prof;
  int prof_pending;
  cudaEvent_t prof_ev[2 * kProfPairs];
  int prof_cls[kProfPairs];
  double prof_ms[kProfClasses];
  long long prof_cnt[kProfClasses];
  char err[256];
};

namespace {

int fail(arche_ctx *c, int code, const char *what, cudaError_t e = cudaSuccess) {
  if (c) snprintf(c->err, sizeof(c->err), "%s%s%s", what, e != cudaSuccess ? ": " : "", e != cudaSuccess ? cudaGetErrorString(e) : "");
  return code;
}
#define CK(call)                                                             \
  do {                                                                       \
    cudaError_t e__ = (call);                                                \
    if (e__ != cudaSuccess) return fail(c, ARCHE_ECUDA, #call, e__);         \
  } while (0)
#define LAUNCHED(c) do { ++(c)->launches; CK(cudaGetLastError()); } while (0)

void prof_harvest(arche_ctx *c) {  // call after a stream synchronise
  for (int k = 0; k < c->prof_pending; ++k) {
    float ms = 0.f;
    if (cudaEventElapsedTime(&ms, c->prof_ev[2 * k], c->prof_ev[2 * k + 1]) == cudaSuccess) {
      c->prof_ms[c->prof_cls[k]] += ms; c->prof_cnt[c->prof_cls[k]] += 1;
    }
  }
  c->prof_pending = 0;
}
struct ProfScope {  // records an event pair around the launches issued in its lifetime
  arche_ctx *c; int k;
  ProfScope(arche_ctx *ctx, int cls) : c(ctx), k(-1) {
    if (!c->prof) return;
    if (c->prof_pending == kProfPairs) { cudaStreamSynchronize(c->stream); prof_harvest(c); }
    k = c->prof_pending++;
    c->prof_cls[k] = cls;
    cudaEventRecord(c->prof_ev[2 * k], c->stream);
  }
  ~ProfScope() { if (k >= 0) cudaEventRecord(c->prof_ev[2 * k + 1], c->stream); }
};

// launch on the context's stream, with programmatic stream serialization when enabled (kernels call pdl_wait())
template <class... KArgs, class... Args>
cudaError_t launch_k(arche_ctx *c, void (*kern)(KArgs...), unsigned grid, unsigned block, size_t smem, Args... args) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(grid); cfg.blockDim = dim3(block); cfg.dynamicSmemBytes = smem; cfg.stream = c->stream;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = at; cfg.numAttrs = c->pdl ? 1 : 0;
  return cudaLaunchKernelEx(&cfg, kern, args...);
}

int fft_tile_blocks(int axis, int n, int nx, int ny, int nz) {
  int L = fft_pick_L(axis, n, nx, ny, nz);
  return axis == 0 ? (int)((long long)ny * nz / L) : (axis == 1 ? nz * (nx / L) : ny * (nx / L));
}

// lays out the workspace; with base == nullptr only sizes it
size_t layout(arche_ctx *c, char *base) {
  Carver w{base, 0};
  const size_t ng = (size_t)c->ng, ni = (size_t)(c->nions > 0 ? c->nions : 1);
  const int nx = c->p.grid[0], ny = c->p.grid[1], nz = c->p.grid[2];
  const size_t nh = (size_t)c->nh;
  c->n_i = w.take<double>(ng); c->n_a = w.take<double>(ng); c->V_i = w.take<double>(ng);
  c->vps = w.take<double>(nh); c->va = w.take<double>(nh);
  c->psp_tab = w.take<double>(c->p.psp == 1 && c->p.psp_nk > 0 ? (size_t)c->p.psp_nk : 1);
  c->nh_i = w.take<double2>(nh); c->nh_a = w.take<double2>(nh); c->vh_ie = w.take<double2>(nh);
  c->S = w.take<double2>(nh); c->S2 = w.take<double2>(nh); c->gh = w.take<double2>(nh); c->gh2 = w.take<double2>(nh);
  c->work = w.take<double2>(nh);
  c->kx = w.take<double>(nx); c->ky = w.take<double>(ny); c->kz = w.take<double>(nz);
  c->kx2 = w.take<double>(nx); c->ky2 = w.take<double>(ny); c->kz2 = w.take<double>(nz);
  c->tw[0] = w.take<double2>(nx); c->tw[1] = w.take<double2>(ny); c->tw[2] = w.take<double2>(nz);
  c->ax_ij = w.take<double2>(ni * nx); c->ax_ji = w.take<double2>(ni * nx);
  c->by_ij = w.take<double2>(ni * ny); c->cz_ij = w.take<double2>(ni * nz);
  c->Z = w.take<double>(ni); c->mass = w.take<double>(ni); c->pos = w.take<double>(3 * ni);
  c->F = w.take<double>(3 * ni); c->F_pp = w.take<double>(3 * ni); c->e_pp = w.take<double>(ni);
  c->vel_tmp = w.take<double>(3 * ni);
  c->pp_part = w.take<double>(6 * ni); c->stress = w.take<double>(64);
  c->F_part = w.take<double>((size_t)c->force_slabs * ni * 3);
  {  // column-resident force kernel: W of the virtual rows beyond ny nz, row tables (1 element when unused)
    const size_t nvp = c->force_ch > 0 ? (size_t)force_vrows_padded(ny, nz) : 1, nrw = (size_t)ny * nz;
    c->force_wb = w.take<double2>(c->force_ch > 0 ? (nvp - nrw) * (size_t)c->P : 1);
    c->force_ri = w.take<int4>(nvp); c->force_rk = w.take<double2>(nvp);
  }
  c->fdtab = w.take<double>(kFdTabDoubles);
  c->partials = w.take<double>((size_t)c->red_blocks * kMaxRed);
  c->counter = w.take<unsigned int>(64);
  c->phase_ns = w.take<unsigned long long>(8);
  c->sc = w.take<DevScalars>(1);
  return w.off;
}

void derive_sizes(arche_ctx *c) {
  const int nx = c->p.grid[0], ny = c->p.grid[1], nz = c->p.grid[2];
  c->ng = (long long)nx * ny * nz;
  c->nxh = nx / 2 + 1;
  c->P = (c->nxh + 7) / 8 * 8;
  c->nh = (long long)c->P * ny * nz;
  c->nions = c->p.n_ions;
  c->ew_grid = (int)((c->ng + 255) / 256 < kEwBlocks ? (c->ng + 255) / 256 : kEwBlocks);
  int rb = c->ew_grid;
  for (int a = 1; a < 3; ++a) { int b = fft_tile_blocks(a, c->p.grid[a], c->P, ny, nz); if (b > rb) rb = b; }
  { int b = fft_real_blocks(nx, ny, nz); if (b > rb) rb = b; }
  long long sfb = ((long long)ny * nz + SF_ROWS - 1) / SF_ROWS * ((c->P + SF_THREADS - 1) / SF_THREADS);
  if (sfb > rb) rb = (int)sfb;
  c->red_blocks = rb + 8 + 2 * kEwBlocks;  // + room for the mu kernel's [2][grid][2] + [grid][6] partials
  const long long rows = (long long)ny * nz;
  c->force_ipt = c->nions >= 1024 ? 4 : (c->nions >= 256 ? 2 : 1);
  const int tiles = (c->nions + FC_THREADS * c->force_ipt - 1) / (FC_THREADS * c->force_ipt);
  int slabs = tiles > 0 ? (148 * 4 + tiles - 1) / tiles : 1;
  if (slabs > rows) slabs = (int)rows;
  if (slabs < 1) slabs = 1;
  c->force_rows_per_slab = (int)((rows + slabs - 1) / slabs);
  c->force_slabs = (int)((rows + c->force_rows_per_slab - 1) / c->force_rows_per_slab);
  c->force_ch = 0;
  if (c->nions >= 256 && !getenv("ARCHE_FORCE_ROWS")) {   // column-resident force kernel (force_cols_kernel)
    // columns per thread: the cost of a (row, ion) is 8 fp64 instructions per column, padded columns included, plus about
    // 30 instruction slots per chunk (fold with b_j c_j, row tables, barrier); measured at 384^3 / 2000 ions: 37.7, 36.8,
    // 34.6, 33.4, 32.0 ms for 13, 17, 20, 25, 33 columns (33 columns: 216 registers, two blocks per SM)
    static const int kCh[5] = {13, 17, 20, 25, 33};
    int best = 0; long long bestcost = 1LL << 60;
    for (int q = 0; q < 5; ++q) {
      const long long cost = (long long)((c->nxh + kCh[q] - 1) / kCh[q]) * (8 * kCh[q] + 30);
      if (cost <= bestcost) { bestcost = cost; best = kCh[q]; }
    }
    if (const char *e = getenv("ARCHE_FORCE_CH")) {   // tuning override
      const int v = atoi(e);
      for (int q = 0; q < 5; ++q) if (v == kCh[q]) best = v;
    }
    c->force_ch = best;
    c->force_chunks = (c->nxh + best - 1) / best;
    const long long vrows = force_vrows_padded(ny, nz);
    const int t128 = (c->nions + FCC_THREADS - 1) / FCC_THREADS, per = t128 * c->force_chunks;
    int z = (148 * (best > 25 ? 2 : 3) * 8 + per - 1) / per;        // about 8 waves of the resident blocks
    if (z > vrows / (4 * FCC_GR)) z = (int)(vrows / (4 * FCC_GR));
    if (z < 1) z = 1;
    c->force_rows_per_slab = (int)((vrows + z - 1) / z);
    c->force_rows_per_slab = (c->force_rows_per_slab + FCC_GR - 1) / FCC_GR * FCC_GR;
    c->force_zslabs = (int)((vrows + c->force_rows_per_slab - 1) / c->force_rows_per_slab);
    c->force_slabs = c->force_zslabs * c->force_chunks;
  }
}

bool params_ok(const arche_params *p) {
  if (!p || p->n_ions < 0 || !(p->kT > 0.0)) return false;
  for (int a = 0; a < 3; ++a)
    if (!grid_ok(p->grid[a]) || !(p->cell[a] > 0.0)) return false;
  if (p->n_ions > 0 && (!p->h_Z || !p->h_mass)) return false;
  if (p->xc < 0 || p->xc > 2) return false;
  if (p->psp != 0 && p->psp != 1) return false;
  if (p->ensemble != 0 && p->ensemble != 1) return false;
  if (p->psp == 1) {   // the table must cover every |k| of the grid
    if (p->psp_nk < 4 || !(p->psp_dk > 0.0) || !p->h_psp_table) return false;
    double k2 = 0.0;
    for (int a = 0; a < 3; ++a) { const double ka = (p->grid[a] / 2) / p->cell[a]; k2 += ka * ka; }
    if (sqrt(k2) > (p->psp_nk - 1) * p->psp_dk) return false;
  }
  return true;
}

}  // namespace

extern "C" size_t arche_workspace_bytes(const arche_params *p) {
  if (!params_ok(p)) return 0;
  arche_ctx tmp;
  memset(&tmp, 0, sizeof(tmp));
  tmp.p = *p;
  derive_sizes(&tmp);
  return layout(&tmp, nullptr);
}

// error text of the last failed arche_scf_init of this thread (the context is destroyed on failure)
static thread_local char g_init_err[256] = "null context";
extern "C" const char *arche_last_error(const arche_ctx *c) { return c ? c->err : g_init_err; }
extern "C" long long arche_launch_count(const arche_ctx *c) { return c ? c->launches : 0; }

extern "C" void arche_destroy(arche_ctx *c) {
  if (!c) return;
  if (c->h_sc) cudaFreeHost(c->h_sc);
  if (c->h_stress) cudaFreeHost(c->h_stress);
  for (int k = 0; k < 2 * kProfPairs; ++k) if (c->prof_ev[k]) cudaEventDestroy(c->prof_ev[k]);
  delete c;
}

// Scratch of arche_fft3d_static: lives in the library image, one copy on every GPU that loads the library, until exit.
// In host code `g_fft3d_static_scratch` is a host-side stand-in, NOT a device address: the address the kernels get is
// the one cudaGetSymbolAddress returns, taken once per device at set-up with that device current.
static __device__ __align__(256) double2 g_fft3d_static_scratch[ARCHE_FFT3D_STATIC_MAX_POINTS];
static double2 *g_fft3d_static_ptr[64];   // per device ordinal; written at set-up (arche_scf_init)
static int fft3d_static_setup(arche_ctx *c) {
  int dev = -1;
  CK(cudaGetDevice(&dev));
  if (dev < 0 || dev >= 64) return fail(c, ARCHE_EINVAL, "device ordinal beyond the static-scratch table");
  if (!g_fft3d_static_ptr[dev]) {
    double2 *ptr = nullptr;
    CK(cudaGetSymbolAddress((void **)&ptr, g_fft3d_static_scratch));
    if (!ptr) return fail(c, ARCHE_ECUDA, "cudaGetSymbolAddress returned a null address for the static FFT scratch");
    g_fft3d_static_ptr[dev] = ptr;
  }
  c->fft_static = g_fft3d_static_ptr[dev];
  return ARCHE_OK;
}

static int init_body(arche_ctx *c, const arche_params *p);

extern "C" int arche_scf_init(const arche_params *p, arche_ctx **out) {
  if (!out) return ARCHE_EINVAL;
  *out = nullptr;
  if (!params_ok(p)) { snprintf(g_init_err, sizeof(g_init_err), "invalid parameters"); return ARCHE_EINVAL; }
  arche_ctx *c = new (std::nothrow) arche_ctx;
  if (!c) return ARCHE_ENOMEM;
  memset(c, 0, sizeof(*c));
  const int rc = init_body(c, p);
  if (rc != ARCHE_OK) {   // nothing leaks on any failure path: the context and its pinned blocks go, the text stays readable
    snprintf(g_init_err, sizeof(g_init_err), "%s", c->err[0] ? c->err : "arche_scf_init failed");
    arche_destroy(c);
    return rc;
  }
  *out = c;
  return ARCHE_OK;
}

static int init_body(arche_ctx *c, const arche_params *p) {
  c->p = *p;
  c->stream = (cudaStream_t)p->stream;
  derive_sizes(c);
  { const char *e = getenv("ARCHE_FFT_GENERIC"); c->use_fast = !(e && e[0] == '1'); }
  {  // fused passes while the iteration's working set (3 real + 4 half-spectrum fields) stays well inside the 126 MB L2
    const char *e = getenv("ARCHE_FUSE");
    const double ws = 24.0 * (double)c->ng + 64.0 * (double)c->nh;
    c->fuse = e ? e[0] == '1' : (ws <= 96.0e6 || (c->ng & 1));
    const char *pe = getenv("ARCHE_PERSIST");
    c->persist = c->fuse && c->use_fast && !(pe && pe[0] == '0');
  }
  size_t need = layout(c, nullptr);
  if (!p->d_workspace || p->workspace_bytes < need || ((uintptr_t)p->d_workspace & 255)) return fail(c, ARCHE_ENOMEM, "workspace missing, too small or not 256-byte aligned");
  layout(c, (char *)p->d_workspace);
  const int nx = p->grid[0], ny = p->grid[1], nz = p->grid[2];
  CK(cudaMallocHost((void **)&c->h_sc, sizeof(DevScalars)));
  CK(cudaMallocHost((void **)&c->h_stress, 64 * sizeof(double)));
  // ---- geometry and constants
  GridGeom &G = c->G;
  G.nx = nx; G.ny = ny; G.nz = nz; G.ng = c->ng; G.nxh = c->nxh; G.P = c->P; G.nh = c->nh;
  G.Lx = p->cell[0]; G.Ly = p->cell[1]; G.Lz = p->cell[2];
  G.vol = G.Lx * G.Ly * G.Lz; G.dV = G.vol / (double)c->ng;
  G.kx = c->kx; G.ky = c->ky; G.kz = c->kz; G.kx2 = c->kx2; G.ky2 = c->ky2; G.kz2 = c->kz2;
  std::vector<double> hZ(c->nions + 1, 0.0);
  c->Q = 0.0;
  for (int j = 0; j < c->nions; ++j) { hZ[j] = p->h_Z[j]; c->Q += hZ[j]; }
  ScfConst &C = c->C;
  C.kT = p->kT; C.cTF = sqrt(2.0) / (ARCHE_PI * ARCHE_PI) * pow(p->kT, 1.5);
  C.Ne = p->n_electrons > 0.0 ? p->n_electrons : c->Q;
  C.vol = G.vol; C.dV = G.dV;
  if (!(C.Ne > 0.0)) return fail(c, ARCHE_EINVAL, "no electrons");
  C.eta0 = fd_half_inverse_host(C.Ne / (G.vol * C.cTF));
  double asum = 0.0;
  for (int j = 0; j < c->nions; ++j)   // alpha_s = 2 pi Z rc^2 (Ashcroft) or Z Du(0) (table, f2)
    asum += p->psp == 1 ? hZ[j] * p->h_psp_table[0] : 2.0 * ARCHE_PI * hZ[j] * p->psp_rc * p->psp_rc;
  C.E_ie0 = C.Ne / G.vol * asum;
  C.xc = p->xc; C.mix_mode = p->mix_mode; C.mix_warmup = p->mix_warmup;
  {  // uniform-gas response chi0 = dn/dmu at Ne/|Omega|; largest single-mode value of More's w (reading A11d)
    const double chi0 = C.cTF * 0.5 * fd_host(0, C.eta0) / p->kT;
    const double Lmax = fmax(G.Lx, fmax(G.Ly, G.Lz)), lam = chi0 * Lmax * Lmax / ARCHE_PI;
    C.mix_w_fixed = p->mix_w_fixed > 0.0 ? p->mix_w_fixed : lam / (1.0 + lam);
    C.mix_mu_tol = p->mix_mu_tol;
    C.chi_floor = p->mix_chi_floor > 0.0 ? p->mix_chi_floor * chi0 : 0.0;
  }
  C.tol_F = p->scf_tol_F; C.tol_dn = p->scf_tol_dn;
  C.q_F = 0.0; C.q_dn = 0.0; C.inv_qF = 0.0; C.inv_vol = 1.0 / G.vol;
  if (p->xc == 1) {  // reading A13: quanta of a PZ81 branch flip at n* = 3/(4 pi)
    const double nstar = 0.75 / ARCHE_PI, den = 1.0 + 1.0529 + 0.3334, ec_hi = -0.1423 / den, ec_lo = -0.048 - 0.0116;
    const double vc_hi = ec_hi * (1.0 + (7.0 / 6.0) * 1.0529 + (4.0 / 3.0) * 0.3334) / den;
    const double vc_lo = -0.048 - 0.0311 / 3.0 + (2.0 * -0.0116 - 0.0020) / 3.0;
    const double eta_star = fd_half_inverse_host(nstar / C.cTF);
    const double chi_star = C.cTF * 0.5 * fd_host(0, eta_star) / p->kT;
    C.q_F = fabs(ec_hi - ec_lo) * nstar * G.dV;
    C.q_dn = chi_star * fabs(vc_hi - vc_lo) * sqrt(G.dV);
    C.inv_qF = 1.0 / C.q_F;
  }
  {  // Ewald alpha (reading A18)
    double rc = 0.5 * fmin(G.Lx, fmin(G.Ly, G.Lz));
    double kc = fmin(nx / (2.0 * G.Lx), fmin(ny / (2.0 * G.Ly), nz / (2.0 * G.Lz)));
    c->alpha = p->ewald_alpha > 0.0 ? p->ewald_alpha : sqrt(ARCHE_PI * kc / rc);
  }
  {  // cooperative grid: all blocks must be co-resident
    int dev = 0, sms = 0, per_sm = 0;
    CK(cudaGetDevice(&dev));
    CK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    // kernels that keep the Fermi-Dirac table (49.5 KB) in dynamic shared memory: opt in on this device
    CK(cudaFuncSetAttribute(mu_solve_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kFdTabBytes));
    CK(cudaFuncSetAttribute(fermi_dirac_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kFdTabBytes));
    CK(cudaFuncSetAttribute(pointwise_r_kernel<LoadReal, StoreVi, true, 4>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kFdTabBytes));
    CK(cudaFuncSetAttribute(pointwise_r_kernel<LoadDensity, StoreNull, true, 4>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kFdTabBytes));
    CK(cudaFuncSetAttribute(pointwise_r_kernel<LoadReal, StoreVi, true, 3>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kFdTabBytes));
    CK(cudaFuncSetAttribute(pointwise_r_kernel<LoadDensity, StoreNull, true, 3>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kFdTabBytes));
    { const char *e = getenv("ARCHE_RBLOCKS"); c->r_blocks = (e && e[0] == '4') ? 4 : 3; }
    // programmatic dependent launch pays where launches are short (measured: 128^3 0.209 -> 0.185 ms per iteration, c3
    // 155 -> 177 MD steps/s, 192^3 +1.4%) and costs ~2% at 384^3, where early-resident blocks of the next kernel take
    // shared memory from the tail of the running one: on by default up to 8 M grid points
    { const char *e = getenv("ARCHE_PDL"); c->pdl = e ? e[0] != '0' : c->ng <= 8000000LL; }
    { const char *e = getenv("ARCHE_LAZY_F"); c->lazy_F = e ? e[0] != '0' : true; }
    { const char *e = getenv("ARCHE_S5_ROWS"); c->s5_rows = e ? e[0] != '0' : true; }
    { const char *e = getenv("ARCHE_SF_TMA"); c->sf_tma = e ? e[0] != '0' : true; }
    { const char *e = getenv("ARCHE_MU_SPLIT"); c->mu_split = e ? e[0] != '0' : true; }
    { const char *e = getenv("ARCHE_MU_REGULAR"); c->mu_regular = e ? e[0] != '0' : true; }
    { const char *e = getenv("ARCHE_MU_COOP_ITERS"); c->mu_coop_iters = e ? atoi(e) : 3; }
    CK(cudaFuncSetAttribute(mu_first_eval_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kFdTabBytes));
    // measured: 384^3 210 -> 172 us (0.67 -> 0.82 of the HBM peak); 256^3 49.5 -> 52.9 us, 192^3 27.5 -> 29.0 us (the register
    // kernel is already at 0.87 there and the extra 2 LP N doubles of shared memory cost a resident block)
    { const char *e = getenv("ARCHE_R2C_TMA"); c->r2c_tma = e ? e[0] != '0' : p->grid[0] >= 384; }
    CK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, mu_solve_kernel, 256, kFdTabBytes));
    // one block per SM while the grid fits the per-thread register cache (cheapest grid barrier), else all co-resident blocks
    if (per_sm < 1) return fail(c, ARCHE_ECUDA, "cooperative kernel cannot be resident");
    c->sm_count = sms;
    const long long cache_pts = (long long)sms * 256 * kMuCache;
    long long blocks = c->ng <= cache_pts ? sms : (long long)sms * (per_sm < 3 ? per_sm : 3);
    const long long want = (c->ng + 255) / 256;
    c->mu_grid = (int)(want < blocks ? want : blocks);
    if (c->mu_grid < 1) return fail(c, ARCHE_ECUDA, "cooperative kernel cannot be resident");
  }
  // ---- per-axis tables: k, k^2, twiddles (long double on the host)
  const int dims[3] = {nx, ny, nz};
  const double Ls[3] = {G.Lx, G.Ly, G.Lz};
  double *dk[3] = {c->kx, c->ky, c->kz}, *dk2[3] = {c->kx2, c->ky2, c->kz2};
  for (int a = 0; a < 3; ++a) {
    const int n = dims[a];
    std::vector<double> k(n), k2(n);
    std::vector<double2> tw(n);
    for (int i = 0; i < n; ++i) {
      int m = i <= n / 2 ? i : i - n;
      k[i] = m / Ls[a]; k2[i] = k[i] * k[i];
      long double ang = -2.0L * 3.14159265358979323846264338327950288L * (long double)i / (long double)n;
      tw[i] = make_double2((double)cosl(ang), (double)sinl(ang));
    }
    CK(cudaMemcpyAsync(dk[a], k.data(), n * sizeof(double), cudaMemcpyHostToDevice, c->stream));
    CK(cudaMemcpyAsync(dk2[a], k2.data(), n * sizeof(double), cudaMemcpyHostToDevice, c->stream));
    CK(cudaMemcpyAsync(c->tw[a], tw.data(), n * sizeof(double2), cudaMemcpyHostToDevice, c->stream));
    CK(cudaStreamSynchronize(c->stream));
    if (!fft_make_plan(n, c->tw[a], &c->plan[a])) return fail(c, ARCHE_EINVAL, "no FFT plan for this axis length");
  }
  if (c->nions > 0) {
    CK(cudaMemcpyAsync(c->Z, p->h_Z, c->nions * sizeof(double), cudaMemcpyHostToDevice, c->stream));
    CK(cudaMemcpyAsync(c->mass, p->h_mass, c->nions * sizeof(double), cudaMemcpyHostToDevice, c->stream));
  }
  std::vector<double> tab(kFdTabDoubles);
  fd_pack_tables(tab.data());
  CK(cudaMemcpyAsync(c->fdtab, tab.data(), kFdTabDoubles * sizeof(double), cudaMemcpyHostToDevice, c->stream));
  CK(cudaMemsetAsync(c->counter, 0, 64 * sizeof(unsigned int), c->stream));
  for (double2 *a : {c->S, c->S2, c->vh_ie, c->gh, c->gh2, c->nh_i, c->nh_a, c->work})   // padding columns stay zero
    CK(cudaMemsetAsync(a, 0, (size_t)c->nh * sizeof(double2), c->stream));
  CK(cudaMemsetAsync(c->sc, 0, sizeof(DevScalars), c->stream));
  CK(cudaMemsetAsync(c->F, 0, 3 * (c->nions > 0 ? c->nions : 1) * sizeof(double), c->stream));
  c->T.on = p->psp == 1 ? 1 : 0; c->T.nk = p->psp_nk; c->T.dk = p->psp_dk; c->T.tab = c->psp_tab;
  if (c->T.on) CK(cudaMemcpyAsync(c->psp_tab, p->h_psp_table, (size_t)p->psp_nk * sizeof(double), cudaMemcpyHostToDevice, c->stream));
  form_factor_kernel<<<c->ew_grid, 256, 0, c->stream>>>(G, p->psp_rc, c->T, c->alpha, c->vps, c->va);
  if (c->force_ch > 0) force_rowinfo_kernel<<<64, 256, 0, c->stream>>>(G, c->force_ri, c->force_rk);
  LAUNCHED(c);
  CK(cudaStreamSynchronize(c->stream));
  c->p.h_Z = nullptr; c->p.h_mass = nullptr; c->p.h_psp_table = nullptr;  // copied; do not keep the caller's pointers
  return fft3d_static_setup(c);
}

// =============================================================================================
// 3D transforms with fused prologue / epilogue
// =============================================================================================
namespace {

// one y or z pass over the half spectrum: register two-stage kernel for the production sizes, generic kernel otherwise
template <int AXIS, bool INVERSE, class LoadOp, class StoreOp>
cudaError_t pass_yz(arche_ctx *c, LoadOp ld, StoreOp st) {
  const int ny = c->G.ny, nz = c->G.nz, P = c->P, n = AXIS == 1 ? ny : nz;
  FastGeom fg{c->G.nx, ny, nz, P, c->tw[AXIS], c->stop, c->pdl ? 1 : 0};
  cudaError_t e = c->use_fast ? fft_launch_yz_fast<AXIS, INVERSE>(n, fg, ld, st, c->stream) : cudaErrorNotSupported;
  if (e == cudaErrorNotSupported) { c->plan[AXIS].stop = c->stop; e = fft_launch_pass<AXIS, INVERSE>(c->plan[AXIS], P, ny, nz, ld, st, c->stream); }
  return e;
}
template <bool INVERSE, class LoadOp, class StoreOp>
cudaError_t pass_x(arche_ctx *c, LoadOp ld, StoreOp st) {
  const int nx = c->G.nx, ny = c->G.ny, nz = c->G.nz, P = c->P;
  FastGeom fg{nx, ny, nz, P, c->tw[0], c->stop, c->pdl ? 1 : 0, c->r2c_tma ? 1 : 0};
  // plain passes of the streamed form run the light configuration (LoadReal / StoreRealPlain / LoadComplex / StoreComplex)
  constexpr bool plain = (std::is_same<LoadOp, LoadReal>::value || std::is_same<LoadOp, LoadComplex>::value) &&
                         (std::is_same<StoreOp, StoreComplex>::value || std::is_same<StoreOp, StoreRealPlain>::value);
  cudaError_t e = cudaErrorNotSupported;
  if (c->use_fast) e = (plain && nx >= 128) ? fft_launch_x_fast<INVERSE, plain>(nx, fg, ld, st, c->stream)
                                            : fft_launch_x_fast<INVERSE, false>(nx, fg, ld, st, c->stream);
  if (e == cudaErrorNotSupported) { c->plan[0].stop = c->stop; e = fft_launch_real_x<INVERSE>(c->plan[0], nx, ny, nz, P, ld, st, c->stream); }
  return e;
}

// inverse (half spectrum -> real field): axis order z, y, x; the x pass is the c2r pass and writes the real field
template <class LoadOp, class StoreOp>
int fft3d_inverse(arche_ctx *c, LoadOp ld, StoreOp st, int cls_first = PC_OTHER, int cls_last = PC_OTHER) {
  { ProfScope ps(c, cls_first);
    CK((pass_yz<2, true>(c, ld, StoreComplex{c->work}))); ++c->launches; }
  { ProfScope ps(c, cls_first == PC_OTHER ? PC_OTHER : PC_FFT_Y);
    CK((pass_yz<1, true>(c, LoadComplex{c->work}, StoreComplex{c->work}))); ++c->launches; }
  { ProfScope ps(c, cls_last);
    CK((pass_x<true>(c, LoadComplex{c->work}, st))); ++c->launches; }
  return ARCHE_OK;
}
// forward (real field -> half spectrum): axis order x (r2c), y, z
template <class LoadOp, class StoreOp>
int fft3d_forward(arche_ctx *c, LoadOp ld, StoreOp st, int cls_first = PC_OTHER, int cls_last = PC_OTHER) {
  { ProfScope ps(c, cls_first);
    CK((pass_x<false>(c, ld, StoreComplex{c->work}))); ++c->launches; }
  { ProfScope ps(c, cls_first == PC_OTHER ? PC_OTHER : PC_FFT_Y);
    CK((pass_yz<1, false>(c, LoadComplex{c->work}, StoreComplex{c->work}))); ++c->launches; }
  { ProfScope ps(c, cls_last);
    CK((pass_yz<2, false>(c, LoadComplex{c->work}, st))); ++c->launches; }
  return ARCHE_OK;
}

int read_scalars(arche_ctx *c) {
  CK(cudaMemcpyAsync(c->h_sc, c->sc, sizeof(DevScalars), cudaMemcpyDeviceToHost, c->stream));
  CK(cudaStreamSynchronize(c->stream));
  if (c->prof) prof_harvest(c);
  return ARCHE_OK;
}

void fill_result(const arche_ctx *c, arche_result *r) {
  if (!r) return;
  const DevScalars &s = *c->h_sc;
  r->mu = s.mu; r->F_total = s.F_total; r->F0 = s.F0; r->E_H = s.EH; r->E_xc = s.Exc; r->E_ie = s.Eie;
  r->E_ie0 = c->C.E_ie0; r->U_ii = s.U_ii; r->K_e = s.Ke; r->K_i = s.K_i; r->dn_l2 = s.dn_rel;
  r->w_last = s.w; r->U_mix = s.U; r->K_mix = s.K; r->tol_F_eff = s.tolF_eff; r->tol_dn_eff = s.toldn_eff;
  r->scf_iters = s.iter; r->mu_evals = s.mu_evals_total; r->converged = s.converged; r->flip_seen = s.flip_seen;
  r->F_evals = s.F_evals;
}

// forward transform of the real input density into nhat_i (scaled by dV)
int input_density_to_g(arche_ctx *c) {
  return fft3d_forward(c, LoadReal{c->n_i}, StoreScaled{c->nh_i, c->G.dV, c->nxh});
}

// applies a pending S6 step to n_i / nhat_i (normally fused into the next iteration's S1/S2 passes)
int flush_mix(arche_ctx *c) {
  if (!c->mix_pending) return ARCHE_OK;
  ProfScope ps(c, PC_MIX);
  mix_kernel<<<c->ew_grid, 256, 0, c->stream>>>(c->n_i, c->n_a, c->nh_i, c->nh_a, c->ng, c->nh, c->sc);
  LAUNCHED(c);
  c->mix_pending = false;
  return ARCHE_OK;
}

static inline bool mu_split_applies(const arche_ctx *c) {
  return c->mu_split && !(c->ng & 1) && c->ng > (long long)c->mu_grid * 256 * kMuCache;
}
// parts: 1 = S1 + S2, 2 = S3 (mu), 4 = S4 + S5.  mu_mode: 0 = first evaluation as an ordinary launch (where it applies),
// then the cooperative kernel; 1 = two ordinary launches and no cooperative one (an iteration they cannot close halts the
// batch: stop flag = 2, scf_solve finishes it); 2 = the cooperative kernel alone
int scf_iteration(arche_ctx *c, int parts = 7, int mu_mode = 0) {
  const GridGeom &G = c->G;
  const ScfConst &C = c->C;
  const int mix = c->mix_pending ? 1 : 0;
  // streaming kernels: up to 16 blocks per SM, but at least 4 half-spectrum elements / 2 real pairs per thread (every
  // block takes part in the closing grid reduction, so an over-sized grid only adds to its tail)
  const int pmax = c->ew_grid * 2;
  auto fit = [&](long long work) { long long b = (work + 255) / 256; return (int)(b < c->sm_count ? c->sm_count : (b > pmax ? pmax : b)); };
  const int pg = fit(c->nh / 4), pr = fit(c->ng / 4);
  // real-space Fermi-Dirac kernels of the streamed form: table in shared memory, co-resident blocks only
  auto prt = [&](int per_sm) { const int b = c->sm_count * per_sm; return pr < b ? pr : b; };
  // S1 + S2 (+ the pending S6 of the previous iteration, + the first mu evaluation)
  LoadPotentialG lp;
  lp.nh_i = c->nh_i; lp.nh_a = c->nh_a; lp.vh_ie = c->vh_ie; lp.kx2 = c->kx2; lp.ky2 = c->ky2; lp.kz2 = c->kz2;
  lp.sc = c->sc; lp.nxh = c->nxh; lp.mix = mix; lp.w = 1.0;
  StoreVi sv;
  sv.V_i = c->V_i; sv.n_i = c->n_i; sv.n_a = c->n_a; sv.sc = c->sc; sv.partials = c->partials; sv.counter = c->counter;
  sv.fdtab = c->fdtab; sv.inv_vol = 1.0 / G.vol; sv.kT_eta0 = C.kT * C.eta0; sv.inv_kT = 1.0 / C.kT; sv.xc = C.xc; sv.mix = mix;
  int rc;
  if (!(parts & 1)) {
  } else if (c->fuse) {
    rc = fft3d_inverse(c, lp, sv, PC_FFT_INV_Z, PC_FFT_INV_X);
    if (rc) return rc;
  } else {
    { ProfScope ps(c, PC_POT_G);
      CK(launch_k(c, pointwise_g_kernel<LoadPotentialG, StoreComplex>, pg, 256, 0, lp, StoreComplex{c->work}, c->P, G.ny, c->nh, c->stop)); ++c->launches; }
    rc = fft3d_inverse(c, LoadComplex{c->work}, StoreRealPlain{c->V_i}, PC_FFT_INV_Z, PC_FFT_INV_X);
    if (rc) return rc;
    { ProfScope ps(c, PC_VI_R);
      if (c->r_blocks == 4) CK(launch_k(c, pointwise_r_kernel<LoadReal, StoreVi, true, 4>, prt(4), 256, kFdTabBytes, LoadReal{c->V_i}, sv, c->ng, c->stop, (const double *)c->fdtab));
      else CK(launch_k(c, pointwise_r_kernel<LoadReal, StoreVi, true, 3>, prt(3), 256, kFdTabBytes, LoadReal{c->V_i}, sv, c->ng, c->stop, (const double *)c->fdtab));
      ++c->launches; }
  }
  if (parts & 1) c->mix_pending = false;
  // S3: persistent cooperative kernel (Newton/secant passes separated by grid barriers)
  if (parts & 2) { ProfScope ps(c, PC_MU);
    const double *aV = c->V_i; long long ang = c->ng; ScfConst aC = C;
    DevScalars *asc = c->sc; const double *atab = c->fdtab; double *apart = c->partials;
    int amax = kMuMaxPasses; const int *astop = c->stop;
    // streamed grids: the one evaluation a steady-state iteration needs as an ordinary dependent launch; the cooperative
    // kernel then returns at once (mu_done) or takes over a hard case
    if (mu_mode != 2 && mu_split_applies(c)) {
      CK(launch_k(c, mu_first_eval_kernel, c->mu_grid, 256, kFdTabBytes, aV, ang, aC, asc, atab, apart, c->counter, astop, 0));
      ++c->launches;
      if (mu_mode == 1) {
        CK(launch_k(c, mu_first_eval_kernel, c->mu_grid, 256, kFdTabBytes, aV, ang, aC, asc, atab, apart, c->counter, astop, 1));
        ++c->launches;
      }
    }
    if (mu_mode != 1 || !mu_split_applies(c)) {
      void *args[] = {&aV, &ang, &aC, &asc, &atab, &apart, &amax, &astop};
      CK(cudaLaunchCooperativeKernel((const void *)mu_solve_kernel, dim3(c->mu_grid), dim3(256), args, kFdTabBytes, c->stream));
      ++c->launches;
    } }
  if (!(parts & 4)) return ARCHE_OK;
  // S4 + S5 (+ w, F, stop flags in the last block of the G-space reduction)
  LoadDensity ldn;
  ldn.V_i = c->V_i; ldn.n_i = c->n_i; ldn.n_a = c->n_a; ldn.sc = c->sc; ldn.partials = c->partials; ldn.counter = c->counter;
  ldn.fdtab = c->fdtab; ldn.C = C;
  StoreNhatA sn;
  sn.nh_a = c->nh_a; sn.nh_i = c->nh_i; sn.vh_ie = c->vh_ie; sn.kx2 = c->kx2; sn.ky2 = c->ky2; sn.kz2 = c->kz2;
  sn.sc = c->sc; sn.partials = c->partials; sn.counter = c->counter; sn.C = C; sn.H.nx = G.nx; sn.H.nxh = c->nxh;
  sn.prestored = c->fuse ? 0 : 1;
  if (c->fuse) {
    rc = fft3d_forward(c, ldn, sn, PC_DENSITY, PC_FFT_FWD_Z);
    if (rc) return rc;
  } else {
    { ProfScope ps(c, PC_DENS_R);
      if (c->r_blocks == 4) CK(launch_k(c, pointwise_r_kernel<LoadDensity, StoreNull, true, 4>, prt(4), 256, kFdTabBytes, ldn, StoreNull{}, c->ng, c->stop, (const double *)c->fdtab));
      else CK(launch_k(c, pointwise_r_kernel<LoadDensity, StoreNull, true, 3>, prt(3), 256, kFdTabBytes, ldn, StoreNull{}, c->ng, c->stop, (const double *)c->fdtab));
      ++c->launches; }
    rc = fft3d_forward(c, LoadReal{c->n_a}, StoreScaled{c->nh_a, G.dV, c->nxh}, PC_FFT_FWD_X, PC_FFT_FWD_Z);
    if (rc) return rc;
    { ProfScope ps(c, PC_RED_G);
      const int nrows = G.ny * G.nz;
      if (c->s5_rows && c->nxh <= 1024) {   // row walk: a thread keeps its kx column, four rows in flight
        const int th = (c->nxh + 31) / 32 * 32 < 256 ? (c->nxh + 31) / 32 * 32 : 256;
        int blocks = c->sm_count * (2048 / th > 8 ? 8 : 2048 / th);
        if (blocks > nrows / 4) blocks = nrows / 4 > 0 ? nrows / 4 : 1;
        const int rpb = (nrows + blocks - 1) / blocks;
        blocks = (nrows + rpb - 1) / rpb;
        CK(launch_k(c, s5_rows_kernel<4>, blocks, th, 0, sn, c->P, G.ny, nrows, rpb, c->stop)); ++c->launches;
      } else {
        CK(launch_k(c, pointwise_g_kernel<LoadComplex, StoreNhatA>, pg, 256, 0, LoadComplex{c->nh_a}, sn, c->P, G.ny, c->nh, c->stop)); ++c->launches;
      } }
  }
  c->mix_pending = true;   // S6 is applied by the next iteration's S1/S2 passes, or by flush_mix()
  c->have_solution = true;
  c->have_forces = false;
  return ARCHE_OK;
}

int scf_begin(arche_ctx *c, const double *d_pos) {
  const GridGeom &G = c->G;
  const int ni = c->nions;
  if (ni > 0) {
    if (!d_pos) return fail(c, ARCHE_EINVAL, "d_pos is null");
    if (d_pos != c->pos) CK(cudaMemcpyAsync(c->pos, d_pos, 3 * ni * sizeof(double), cudaMemcpyDeviceToDevice, c->stream));
    // P1: separable phase tables, then S_Z with the V_ie / Ewald-reciprocal epilogue (P2, P3)
    const int pb = 148 * 2;
    phase_table_kernel<<<pb, 256, 0, c->stream>>>(c->pos, 0, G.Lx, G.nx, ni, c->ax_ij, c->ax_ji); LAUNCHED(c);
    phase_table_kernel<<<pb, 256, 0, c->stream>>>(c->pos, 1, G.Ly, G.ny, ni, c->by_ij, nullptr); LAUNCHED(c);
    phase_table_kernel<<<pb, 256, 0, c->stream>>>(c->pos, 2, G.Lz, G.nz, ni, c->cz_ij, nullptr); LAUNCHED(c);
    { ProfScope ps(c, PC_SFAC);
    // register-tiled kernel when nx/2 splits into IXT columns per thread with whole warps, else the generic one
    const int nxm = G.nx / 2;
    const int ixt = (G.nx % 2 == 0 && ni >= 256) ? (nxm % 128 == 0 ? 4 : (nxm % 96 == 0 ? 3 : (nxm % 64 == 0 ? 2 : 0))) : 0;
    int own_nyq_x = 0;
    const int txb_t = ixt ? nxm / ixt : 0, rg_t = txb_t ? 128 / txb_t : 0;
    const bool tma_ok = c->sf_tma && ixt && txb_t * rg_t == 128 &&
                        ((ixt == 3 && rg_t == 2) || (ixt == 4 && rg_t == 4) || (ixt == 3 && rg_t == 4) || (ixt == 2 && rg_t == 4));
    if (tma_ok) {   // register tile fed by the copy engine (structure_factor_tma_kernel)
      const unsigned blocks = (unsigned)(((long long)G.ny * G.nz + SF2_ROWS * rg_t - 1) / (SF2_ROWS * rg_t));
      const size_t smem = ((size_t)SF3_NST * SF3_JT * nxm + 2 * (size_t)SF2_ROWS * rg_t * SF3_JT) * sizeof(double2);
#define ARCHE_SFT(I, R) { auto kern = structure_factor_tma_kernel<I, R>; \
        CK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem)); \
        kern<<<blocks, 128, smem, c->stream>>>(G, ni, c->Z, c->ax_ji, c->by_ij, c->cz_ij, c->vps, c->va, c->S, c->S2, c->vh_ie, c->partials, c->counter, c->sc); }
      if (ixt == 3 && rg_t == 2) ARCHE_SFT(3, 2) else if (ixt == 4) ARCHE_SFT(4, 4) else if (ixt == 3) ARCHE_SFT(3, 4) else ARCHE_SFT(2, 4)
#undef ARCHE_SFT
      own_nyq_x = 1;
    } else if (ixt) {
      const unsigned blocks = (unsigned)(((long long)G.ny * G.nz + SF2_ROWS - 1) / SF2_ROWS);
      const int txb = nxm / ixt;
      if (ixt == 4) structure_factor_tiled_kernel<4><<<blocks, txb, 0, c->stream>>>(G, ni, c->Z, c->ax_ji, c->by_ij, c->cz_ij, c->vps, c->va, c->S, c->S2, c->vh_ie, c->partials, c->counter, c->sc);
      else if (ixt == 3) structure_factor_tiled_kernel<3><<<blocks, txb, 0, c->stream>>>(G, ni, c->Z, c->ax_ji, c->by_ij, c->cz_ij, c->vps, c->va, c->S, c->S2, c->vh_ie, c->partials, c->counter, c->sc);
      else structure_factor_tiled_kernel<2><<<blocks, txb, 0, c->stream>>>(G, ni, c->Z, c->ax_ji, c->by_ij, c->cz_ij, c->vps, c->va, c->S, c->S2, c->vh_ie, c->partials, c->counter, c->sc);
      own_nyq_x = 1;
    } else {
      dim3 sg((unsigned)(((long long)G.ny * G.nz + SF_ROWS - 1) / SF_ROWS), (unsigned)((c->P + SF_THREADS - 1) / SF_THREADS));
      structure_factor_kernel<<<sg, SF_THREADS, 0, c->stream>>>(G, ni, c->Z, c->ax_ji, c->by_ij, c->cz_ij, c->vps, c->va, c->S,
                                                                c->S2, c->vh_ie, c->partials, c->counter, c->sc);
    }
    LAUNCHED(c);
    structure_factor_nyquist_kernel<<<c->ew_grid, 128, 0, c->stream>>>(G, ni, c->Z, c->ax_ij, c->by_ij, c->cz_ij, c->vps, c->va,
                                                                       c->S, c->S2, c->vh_ie, c->partials, c->counter, c->sc, own_nyq_x);
    LAUNCHED(c); }
    ewald_pp_kernel<<<ni, 128, 0, c->stream>>>(c->pos, c->Z, ni, G.Lx, G.Ly, G.Lz, c->alpha, c->F_pp, c->e_pp); LAUNCHED(c);
    ewald_finish_kernel<<<1, 256, 0, c->stream>>>(c->e_pp, c->Z, ni, c->alpha, G.vol, c->sc); LAUNCHED(c);
  } else {
    CK(cudaMemsetAsync(c->S, 0, c->nh * sizeof(double2), c->stream));
    CK(cudaMemsetAsync(c->S2, 0, c->nh * sizeof(double2), c->stream));
    CK(cudaMemsetAsync(c->vh_ie, 0, c->nh * sizeof(double2), c->stream));
  }
  // P4: input density
  if (c->p.init_mode == 1 && c->have_g && ni > 0) {
    StoreClip sk;
    sk.n_i = c->n_i; sk.sc = c->sc; sk.partials = c->partials; sk.counter = c->counter;
    sk.inv_vol = 1.0 / G.vol; sk.floor_n = 1e-3 * c->C.Ne / G.vol; sk.Ne = c->C.Ne; sk.dV = G.dV; sk.acc = 0.0;
    int rc = fft3d_inverse(c, LoadSG{c->S, c->S2, c->gh, c->gh2, c->nxh}, sk);
    if (rc) return rc;
    rc = fft3d_forward(c, LoadRealScaled{c->n_i, c->sc, 1.0}, StoreScaled{c->nh_i, G.dV, c->nxh});
    if (rc) return rc;
    c->C.mix_warmup = 0;  // profile start: mu fluctuations are small from the first iteration (reading A11)
  } else {
    c->C.mix_warmup = c->p.mix_warmup;
    set_uniform_kernel<<<c->ew_grid, 256, 0, c->stream>>>(c->n_i, c->nh_i, c->ng, c->nh, c->C.Ne / G.vol, c->C.Ne);
    LAUNCHED(c);
  }
  // reset per-solve scalars (iter, F_total, converged); mu and U_ii persist
  CK(cudaMemsetAsync(&c->sc->iter, 0, sizeof(int) * 6, c->stream));   // iter, converged, mu_evals_total, flip_seen, more_on, pad
  CK(cudaMemsetAsync(&c->sc->F_total, 0, sizeof(double), c->stream));
  CK(cudaMemsetAsync(&c->sc->mu_evals_total, 0, sizeof(int), c->stream));
  CK(cudaMemsetAsync(&c->sc->skip_F, 0, 4 * sizeof(int), c->stream));   // skip_F, F_valid, F_evals, pad
  c->C.lazy_F = 0;   // the split form (arche_scf_iter) evaluates the free energy in every iteration
  c->have_solution = false;
  c->have_forces = false;
  c->mix_pending = false;  // a new input density replaces any unapplied mixing step
  return ARCHE_OK;
}

int scf_solve(arche_ctx *c, const double *d_pos) {
  int rc = scf_begin(c, d_pos);
  if (rc) return rc;
  const int fixed = c->p.scf_fixed_iter;
  const int maxit = fixed > 0 ? fixed : (c->p.scf_max_iter > 0 ? c->p.scf_max_iter : 200);
  bool conv = false;
  // lazy free energy (ScfConst::lazy_F): under the stop rule F is evaluated only where the rule can use it.  Not with the
  // printed PZ81 constants (the branch-flip detection of reading A13 watches F in every iteration), not in parity replays.
  c->C.lazy_F = (fixed <= 0 && c->p.xc != 1 && c->lazy_F) ? maxit : 0;
  // L2-resident production grids: the whole solve in one cooperative launch (with per-class profiling on, block 0
  // times the phases with %globaltimer and the classes receive those times)
  if (c->persist) {
    PersistParams pp;
    pp.phase_ns = c->prof ? c->phase_ns : nullptr;
    if (c->prof) CK(cudaMemsetAsync(c->phase_ns, 0, 8 * sizeof(unsigned long long), c->stream));
    pp.n_i = c->n_i; pp.n_a = c->n_a; pp.V_i = c->V_i; pp.nh_i = c->nh_i; pp.nh_a = c->nh_a; pp.work = c->work;
    pp.vh_ie = c->vh_ie; pp.kx2 = c->kx2; pp.ky2 = c->ky2; pp.kz2 = c->kz2;
    pp.tw0 = c->tw[0]; pp.tw1 = c->tw[1]; pp.tw2 = c->tw[2];
    pp.sc = c->sc; pp.partials = c->partials; pp.counter = c->counter; pp.fdtab = c->fdtab; pp.C = c->C;
    pp.nxh = c->nxh; pp.P = c->P; pp.ng = c->ng; pp.inv_vol = 1.0 / c->G.vol;
    pp.mix_first = c->mix_pending ? 1 : 0; pp.max_iters = maxit; pp.fixed = fixed > 0 ? 1 : 0; pp.mu_max_pass = kMuMaxPasses;
    cudaError_t e = scf_persistent_launch(c->G.nx, c->G.ny, c->G.nz, pp, c->sm_count * kPersistBlocksPerSM, c->stream);
    if (e == cudaSuccess) {
      ++c->launches;
      c->mix_pending = true; c->have_solution = true; c->have_forces = false;
      rc = read_scalars(c);
      if (rc) return rc;
      if (c->prof) {
        unsigned long long ns[8];
        CK(cudaMemcpy(ns, c->phase_ns, sizeof(ns), cudaMemcpyDeviceToHost));
        const int cls[7] = {PC_FFT_INV_Z, PC_FFT_Y, PC_FFT_INV_X, PC_MU, PC_DENSITY, PC_FFT_Y, PC_FFT_FWD_Z};
        for (int k = 0; k < 7; ++k) { c->prof_ms[cls[k]] += 1e-6 * (double)ns[k]; c->prof_cnt[cls[k]] += (long long)ns[7]; }
      }
      if (!isfinite(c->h_sc->F_total) || !isfinite(c->h_sc->mu)) return fail(c, ARCHE_ENAN, "non-finite free energy or mu");
      conv = fixed <= 0 && c->h_sc->converged;
      goto solved;
    }
    if (e == cudaErrorCooperativeLaunchTooLarge) (void)cudaGetLastError();   // GPU shared with another context: per-pass form
    else if (e != cudaErrorNotSupported) return fail(c, ARCHE_ECUDA, "scf_persistent_launch", e);
    c->persist = false;   // no instantiation for this grid (or no room for the resident grid): per-pass form from now on
  }
  // Iterations are launched in batches without a host round trip; once the S5 epilogue has set the stop flag the
  // kernels of the remaining iterations of the batch return at once, so the state stays that of the converged
  // iteration.  Parity replays (scf_fixed_iter) run every iteration.
  {
  // The batch length follows the residual: from the contraction of ||dn|| over the last batch the host predicts how
  // many iterations are left and launches that many (1 ... 2 kScfBatch) -- fewer host round trips early in the solve,
  // no tail of no-op launches at its end (at 128^3 an iteration is 11 launches of 12-25 us; the fixed batch of six left
  // 2.5 iterations of no-ops per solve on average, 1.3% of the c3 MD step).
  int batch = fixed > 0 ? maxit : kScfBatch;
  double dn_prev = 0.0;
  for (int it = 0; it < maxit && !conv;) {
    c->stop = fixed > 0 ? nullptr : &c->sc->converged;
    const int n = it + batch <= maxit ? batch : maxit - it;
    for (int b = 0; b < n; ++b) {
      // after the first iterations of a solve (no previous mu, large steps) the mu iteration runs as ordinary launches only
      const int mode = (fixed <= 0 && c->mu_regular && mu_split_applies(c) && it + b >= c->mu_coop_iters) ? 1 : 0;
      rc = scf_iteration(c, 7, mode);
      if (rc) { c->stop = nullptr; return rc; }
    }
    rc = read_scalars(c);
    if (rc) { c->stop = nullptr; return rc; }
    if (fixed <= 0 && c->h_sc->converged == 2) {
      // an iteration whose mu the ordinary launches could not close halted the batch (every later kernel returned at
      // once): the cooperative kernel takes over from the handed-over state, then the rest of that iteration runs
      CK(cudaMemsetAsync(&c->sc->converged, 0, sizeof(int), c->stream));
      rc = scf_iteration(c, 2 | 4, 2);
      if (rc) { c->stop = nullptr; return rc; }
      rc = read_scalars(c);
      if (rc) { c->stop = nullptr; return rc; }
    }
    c->stop = nullptr;
    const int it_before = it;
    it = fixed > 0 ? it + n : c->h_sc->iter;   // the device's count: a halted batch completed fewer iterations than launched
    const int n_done = it > it_before ? it - it_before : 1;
    if (!isfinite(c->h_sc->F_total) || !isfinite(c->h_sc->mu)) return fail(c, ARCHE_ENAN, "non-finite free energy or mu");
    if (fixed <= 0 && c->h_sc->converged) conv = true;
    if (fixed <= 0 && !conv) {
      const double dn = c->h_sc->dn_rel, tol = c->h_sc->toldn_eff;
      batch = kScfBatch;
      if (dn > 0.0 && tol > 0.0) {
        if (dn <= tol) batch = 1;                                  // waiting for the free-energy criterion only
        else if (dn_prev > dn) {
          const double rem = log(tol / dn) * (double)n_done / log(dn / dn_prev);   // iterations until ||dn|| meets the tolerance
          batch = rem < 1.0 ? 1 : (rem > 2.0 * kScfBatch ? 2 * kScfBatch : (int)ceil(rem));
        }
      }
      dn_prev = dn;
    }
  }
  }
solved:
  c->C.lazy_F = 0;
  // P6: one-center profile of this step's converged density (reading A10)
  if (c->nions > 0) {
    g_store_kernel<<<c->ew_grid, 256, 0, c->stream>>>(c->gh, c->gh2, c->nh_a, c->S, c->S2, c->nh, 1e-8 * c->Q * c->Q);
    LAUNCHED(c);
    c->have_g = true;
  }
  return (conv || fixed > 0) ? ARCHE_OK : fail(c, ARCHE_ENOCONV, "SCF did not converge within scf_max_iter");
}

int compute_forces(arche_ctx *c) {
  if (!c->have_solution) return fail(c, ARCHE_EINVAL, "arche_forces before a solve");
  const int ni = c->nions;
  if (ni == 0) { c->have_forces = true; return ARCHE_OK; }
  const GridGeom &G = c->G;
  const int ipt = c->force_ipt, per_block = FC_THREADS * ipt;
  dim3 fg((unsigned)((ni + per_block - 1) / per_block), (unsigned)c->force_slabs);
  const size_t fsm = FC_RPT * c->nxh * sizeof(double2) + c->nxh * sizeof(double);
  { ProfScope ps(c, PC_FORCE);
  if (c->force_ch > 0) {
    dim3 cg((unsigned)((ni + FCC_THREADS - 1) / FCC_THREADS), (unsigned)c->force_chunks, (unsigned)c->force_zslabs);
    force_w_kernel<<<c->ew_grid, 256, 0, c->stream>>>(G, c->vps, c->va, c->nh_a, c->S, c->S2, c->work, c->force_wb); LAUNCHED(c);
#define ARCHE_FCC(CH) force_cols_kernel<CH><<<cg, FCC_THREADS, 0, c->stream>>>(G, ni, c->force_rows_per_slab, c->ax_ij, c->by_ij, \
                                                                       c->cz_ij, c->work, c->force_wb, c->force_ri, c->force_rk, c->F_part)
    if (c->force_ch == 13) ARCHE_FCC(13); else if (c->force_ch == 17) ARCHE_FCC(17); else if (c->force_ch == 20) ARCHE_FCC(20); else if (c->force_ch == 33) ARCHE_FCC(33); else ARCHE_FCC(25);
#undef ARCHE_FCC
  } else if (ipt == 4)
    force_kernel<4><<<fg, FC_THREADS, fsm, c->stream>>>(G, ni, c->force_rows_per_slab, c->ax_ij, c->by_ij, c->cz_ij, c->vps, c->va,
                                                        c->nh_a, c->S, c->S2, c->F_part);
  else if (ipt == 2)
    force_kernel<2><<<fg, FC_THREADS, fsm, c->stream>>>(G, ni, c->force_rows_per_slab, c->ax_ij, c->by_ij, c->cz_ij, c->vps, c->va,
                                                        c->nh_a, c->S, c->S2, c->F_part);
  else
    force_kernel<1><<<fg, FC_THREADS, fsm, c->stream>>>(G, ni, c->force_rows_per_slab, c->ax_ij, c->by_ij, c->cz_ij, c->vps, c->va,
                                                        c->nh_a, c->S, c->S2, c->F_part);
  LAUNCHED(c); }
  force_finish_kernel<<<(3 * ni * 32 + 127) / 128, 128, 0, c->stream>>>(ni, c->force_slabs, c->F_part, c->F_pp, c->Z,
                                                                   -2.0 * ARCHE_PI / G.vol, c->F);
  LAUNCHED(c);
  c->have_forces = true;
  return ARCHE_OK;
}

// f1: stress tensor and pressure of the last solve (stress_kernels.cuh): 3 launches (2 without ions)
int compute_stress(arche_ctx *c, const double *d_vel) {
  if (!c->have_solution) return fail(c, ARCHE_EINVAL, "arche_stress before a solve");
  const int ni = c->nions;
  const GridGeom &G = c->G;
  const long long work = c->nh > c->ng ? c->nh : c->ng;
  long long nb = (work + kStressThreads - 1) / kStressThreads;
  const long long cap = (long long)c->red_blocks * kMaxRed / kStressSums, full = (long long)c->sm_count * 8;
  if (nb > full) nb = full;
  if (nb > cap) nb = cap;
  { ProfScope ps(c, PC_STRESS);
  stress_fields_kernel<<<(unsigned)nb, kStressThreads, 0, c->stream>>>(G, c->nh_a, c->S, c->S2, c->n_a, c->p.xc, c->alpha,
                                                                     c->p.psp_rc, c->T, c->partials);
  LAUNCHED(c); }
  if (ni > 0) {
    stress_pp_kernel<<<ni, 128, 0, c->stream>>>(c->pos, c->Z, ni, G.Lx, G.Ly, G.Lz, c->alpha, c->pp_part);
    LAUNCHED(c);
  }
  const StressConst K{G.vol, G.dV, c->alpha, c->Q, c->C.E_ie0};
  stress_finish_kernel<<<1, kStressThreads, 0, c->stream>>>((int)nb, c->partials, ni, c->pp_part, d_vel, c->mass, c->sc, K, c->stress);
  LAUNCHED(c);
  return ARCHE_OK;
}

}  // namespace

// =============================================================================================
// C ABI
// =============================================================================================
extern "C" int arche_scf_begin(arche_ctx *c, const double *d_pos) {
  if (!c) return ARCHE_EINVAL;
  return scf_begin(c, d_pos);
}

extern "C" int arche_scf_iter(arche_ctx *c, arche_result *h_out) {
  if (!c) return ARCHE_EINVAL;
  int rc = scf_iteration(c);
  if (rc) return rc;
  rc = read_scalars(c);
  if (rc) return rc;
  fill_result(c, h_out);
  return ARCHE_OK;
}

extern "C" int arche_set_input_density(arche_ctx *c, const double *d_n) {
  if (!c || !d_n) return ARCHE_EINVAL;
  CK(cudaMemcpyAsync(c->n_i, d_n, c->ng * sizeof(double), cudaMemcpyDeviceToDevice, c->stream));
  c->mix_pending = false;
  return input_density_to_g(c);
}

extern "C" int arche_scf_solve(arche_ctx *c, const double *d_pos, arche_result *h_out) {
  if (!c) return ARCHE_EINVAL;
  int rc = scf_solve(c, d_pos);
  if (rc != ARCHE_OK && rc != ARCHE_ENOCONV) return rc;
  int r2 = read_scalars(c);
  if (r2) return r2;
  fill_result(c, h_out);
  return rc;
}

extern "C" int arche_forces(arche_ctx *c, double *d_F) {
  if (!c) return ARCHE_EINVAL;
  int rc = compute_forces(c);
  if (rc) return rc;
  if (d_F && c->nions > 0) CK(cudaMemcpyAsync(d_F, c->F, 3 * c->nions * sizeof(double), cudaMemcpyDeviceToDevice, c->stream));
  return ARCHE_OK;
}

extern "C" int arche_stress(arche_ctx *c, const double *d_vel, double *h_out) {
  if (!c || !h_out) return ARCHE_EINVAL;
  int rc = compute_stress(c, d_vel);
  if (rc) return rc;
  CK(cudaMemcpyAsync(c->h_stress, c->stress, kStressOut * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
  CK(cudaStreamSynchronize(c->stream));
  if (c->prof) prof_harvest(c);
  memcpy(h_out, c->h_stress, kStressOut * sizeof(double));
  return ARCHE_OK;
}

extern "C" int arche_md_step(arche_ctx *c, double dt, double *d_pos, double *d_vel, arche_result *h_out) {
  if (!c || !d_pos || !d_vel || c->nions <= 0) return ARCHE_EINVAL;
  const int ni = c->nions, nb = (3 * ni + 127) / 128;
  int rc, rc_first = ARCHE_OK;
  if (!c->have_forces) {  // forces at the starting positions
    rc_first = scf_solve(c, d_pos);
    if (rc_first != ARCHE_OK && rc_first != ARCHE_ENOCONV) return rc_first;
    rc = compute_forces(c);
    if (rc) return rc;
  }
  if (c->p.ensemble == 1) { isokinetic_kick_kernel<<<1, 1024, 0, c->stream>>>(d_pos, d_vel, c->F, c->mass, 0.5 * dt, dt, ni, 1); LAUNCHED(c); }
  else { kick_drift_kernel<<<nb, 128, 0, c->stream>>>(d_pos, d_vel, c->F, c->mass, dt, ni, 1); LAUNCHED(c); }
  int rc_solve = scf_solve(c, d_pos);
  if (rc_solve != ARCHE_OK && rc_solve != ARCHE_ENOCONV) return rc_solve;
  rc = compute_forces(c);
  if (rc) return rc;
  if (c->p.ensemble == 1) { isokinetic_kick_kernel<<<1, 1024, 0, c->stream>>>(d_pos, d_vel, c->F, c->mass, 0.5 * dt, dt, ni, 0); LAUNCHED(c); }
  else { kick_drift_kernel<<<nb, 128, 0, c->stream>>>(d_pos, d_vel, c->F, c->mass, dt, ni, 0); LAUNCHED(c); }
  kinetic_kernel<<<1, 256, 0, c->stream>>>(d_vel, c->mass, ni, c->sc); LAUNCHED(c);
  rc = read_scalars(c);
  if (rc) return rc;
  fill_result(c, h_out);
  return rc_solve != ARCHE_OK ? rc_solve : rc_first;   // a non-converged solve at the starting positions is reported too
}

extern "C" int arche_md_step_host(arche_ctx *c, double dt, double *h_pos, double *h_vel, double *h_F, arche_result *h_out) {
  if (!c || !h_pos || !h_vel || c->nions <= 0) return ARCHE_EINVAL;
  const size_t nb = 3 * (size_t)c->nions * sizeof(double);
  // c->pos doubles as the device position buffer; velocities go through vel_tmp
  CK(cudaMemcpyAsync(c->pos, h_pos, nb, cudaMemcpyHostToDevice, c->stream));
  CK(cudaMemcpyAsync(c->vel_tmp, h_vel, nb, cudaMemcpyHostToDevice, c->stream));
  int rc = arche_md_step(c, dt, c->pos, c->vel_tmp, h_out);
  if (rc != ARCHE_OK && rc != ARCHE_ENOCONV) return rc;
  CK(cudaMemcpyAsync(h_pos, c->pos, nb, cudaMemcpyDeviceToHost, c->stream));
  CK(cudaMemcpyAsync(h_vel, c->vel_tmp, nb, cudaMemcpyDeviceToHost, c->stream));
  if (h_F) CK(cudaMemcpyAsync(h_F, c->F, nb, cudaMemcpyDeviceToHost, c->stream));
  CK(cudaStreamSynchronize(c->stream));
  return rc;
}

extern "C" int arche_get_real(arche_ctx *c, int which, double *d_dst) {
  if (!c || !d_dst) return ARCHE_EINVAL;
  const double *src = which == 0 ? c->n_a : which == 1 ? c->n_i : which == 2 ? c->V_i : nullptr;
  if (!src) return ARCHE_EINVAL;
  if (which == 1) { int rc = flush_mix(c); if (rc) return rc; }
  CK(cudaMemcpyAsync(d_dst, src, c->ng * sizeof(double), cudaMemcpyDeviceToDevice, c->stream));
  return ARCHE_OK;
}
extern "C" int arche_get_complex(arche_ctx *c, int which, double *d_dst) {
  if (!c || !d_dst) return ARCHE_EINVAL;
  // the library keeps half spectra; the read-back is the full [nz][ny][nx] array on the literal index set of P:142
  const double2 *src, *src2; const double *scale = nullptr;
  switch (which) {
    case 0: src = src2 = c->nh_a; break;
    case 1: src = c->S; src2 = c->S2; scale = c->vps; break;   // Vhat_ie = v(k) S_Z(k)
    case 2: src = c->S; src2 = c->S2; break;
    case 3: src = c->gh; src2 = c->gh2; break;
    case 4: { int rc = flush_mix(c); if (rc) return rc; src = src2 = c->nh_i; break; }
    default: return ARCHE_EINVAL;
  }
  expand_half_kernel<<<c->ew_grid, 256, 0, c->stream>>>((double2 *)d_dst, src, src2, scale, c->G.nx, c->G.ny, c->G.nz, c->P);
  LAUNCHED(c);
  return ARCHE_OK;
}
extern "C" int arche_get_density(arche_ctx *c, double *d_n) { return arche_get_real(c, 0, d_n); }

extern "C" int arche_fft3d(arche_ctx *c, const double *d_in, double *d_out, double *d_scratch, int sign) {
  if (!c || !d_in || !d_out || !d_scratch || (sign != 1 && sign != -1)) return ARCHE_EINVAL;
  const int nx = c->G.nx, ny = c->G.ny, nz = c->G.nz;
  for (int a = 0; a < 3; ++a) c->plan[a].stop = nullptr;
  double2 *w = (double2 *)d_scratch, *o = (double2 *)d_out;
  const double2 *in = (const double2 *)d_in;
  if (sign < 0) {
    CK((fft_launch_pass<0, false>(c->plan[0], nx, ny, nz, LoadComplex{in}, StoreComplex{w}, c->stream))); ++c->launches;
    CK((fft_launch_pass<1, false>(c->plan[1], nx, ny, nz, LoadComplex{w}, StoreComplex{w}, c->stream))); ++c->launches;
    CK((fft_launch_pass<2, false>(c->plan[2], nx, ny, nz, LoadComplex{w}, StoreComplex{o}, c->stream))); ++c->launches;
  } else {
    CK((fft_launch_pass<2, true>(c->plan[2], nx, ny, nz, LoadComplex{in}, StoreComplex{w}, c->stream))); ++c->launches;
    CK((fft_launch_pass<1, true>(c->plan[1], nx, ny, nz, LoadComplex{w}, StoreComplex{w}, c->stream))); ++c->launches;
    CK((fft_launch_pass<0, true>(c->plan[0], nx, ny, nz, LoadComplex{w}, StoreComplex{o}, c->stream))); ++c->launches;
  }
  return ARCHE_OK;
}

// f4: slab-decomposed complex transform (fft.cuh StoreSlabScatter).  Phase 1 runs the passes before the transpose, the
// last of them storing into the peers' slabs; phase 2, after every rank's phase 1 has completed, the passes after it.
extern "C" int arche_fft3d_slab_scatter(arche_ctx *c, const double *d_in, double *d_scratch, double *const *h_peer,
                                        int n_ranks, int rank, int sign) {
  if (!c || !d_in || !h_peer || (sign != 1 && sign != -1)) return ARCHE_EINVAL;
  const int nx = c->G.nx, ny = c->G.ny, nz = c->G.nz;
  if (n_ranks < 1 || n_ranks > kSlabMaxRanks || rank < 0 || rank >= n_ranks || ny % n_ranks || nz % n_ranks)
    return fail(c, ARCHE_EINVAL, "arche_fft3d_slab: Ny and Nz must be multiples of n_ranks <= 16");
  const int nyl = ny / n_ranks, nzl = nz / n_ranks;
  for (int a = 0; a < 3; ++a) c->plan[a].stop = nullptr;
  StoreSlabScatter st;
  for (int q = 0; q < kSlabMaxRanks; ++q) st.peer[q] = q < n_ranks ? (double2 *)h_peer[q] : nullptr;
  for (int q = 0; q < n_ranks; ++q) if (!h_peer[q]) return ARCHE_EINVAL;
  st.nx = nx;
  const double2 *in = (const double2 *)d_in;
  if (sign < 0) {   // z slab [nzl][ny][nx]: x pass, then the y pass that scatters into the y slabs [nz][nyl][nx]
    if (!d_scratch) return ARCHE_EINVAL;
    double2 *w = (double2 *)d_scratch;
    st.nloc_dst = nyl; st.pitch_dst = nyl; st.off_src = rank * nzl; st.forward = 1;
    CK((fft_launch_pass<0, false>(c->plan[0], nx, ny, nzl, LoadComplex{in}, StoreComplex{w}, c->stream))); ++c->launches;
    CK((fft_launch_pass<1, false>(c->plan[1], nx, ny, nzl, LoadComplex{w}, st, c->stream))); ++c->launches;
  } else {          // y slab [nz][nyl][nx]: the z pass scatters into the z slabs [nzl][ny][nx]
    st.nloc_dst = nzl; st.pitch_dst = ny; st.off_src = rank * nyl; st.forward = 0;
    CK((fft_launch_pass<2, true>(c->plan[2], nx, nyl, nz, LoadComplex{in}, st, c->stream))); ++c->launches;
  }
  return ARCHE_OK;
}

extern "C" int arche_fft3d_slab_finish(arche_ctx *c, double *d_slab, int n_ranks, int sign) {
  if (!c || !d_slab || (sign != 1 && sign != -1)) return ARCHE_EINVAL;
  const int nx = c->G.nx, ny = c->G.ny, nz = c->G.nz;
  if (n_ranks < 1 || n_ranks > kSlabMaxRanks || ny % n_ranks || nz % n_ranks)
    return fail(c, ARCHE_EINVAL, "arche_fft3d_slab: Ny and Nz must be multiples of n_ranks <= 16");
  for (int a = 0; a < 3; ++a) c->plan[a].stop = nullptr;
  double2 *s = (double2 *)d_slab;
  if (sign < 0) {   // y slab: z pass in place
    CK((fft_launch_pass<2, false>(c->plan[2], nx, ny / n_ranks, nz, LoadComplex{s}, StoreComplex{s}, c->stream))); ++c->launches;
  } else {          // z slab: y and x passes in place
    CK((fft_launch_pass<1, true>(c->plan[1], nx, ny, nz / n_ranks, LoadComplex{s}, StoreComplex{s}, c->stream))); ++c->launches;
    CK((fft_launch_pass<0, true>(c->plan[0], nx, ny, nz / n_ranks, LoadComplex{s}, StoreComplex{s}, c->stream))); ++c->launches;
  }
  return ARCHE_OK;
}

// slab buffers that other processes can map: plain cudaMalloc allocations (an IPC handle names a whole allocation,
// so these do not come out of a caching allocator's pool)
extern "C" int arche_slab_alloc(size_t bytes, void **d_out) {
  if (!d_out || bytes == 0) return ARCHE_EINVAL;
  *d_out = nullptr;
  return cudaMalloc(d_out, bytes) == cudaSuccess ? ARCHE_OK : ARCHE_ENOMEM;
}
extern "C" int arche_slab_free(void *d_ptr) { return cudaFree(d_ptr) == cudaSuccess ? ARCHE_OK : ARCHE_ECUDA; }
extern "C" int arche_ipc_export(const void *d_ptr, unsigned char *h_handle64) {
  if (!d_ptr || !h_handle64) return ARCHE_EINVAL;
  cudaIpcMemHandle_t h;
  static_assert(sizeof(h) == 64, "cudaIpcMemHandle_t is 64 bytes");
  if (cudaIpcGetMemHandle(&h, const_cast<void *>(d_ptr)) != cudaSuccess) { (void)cudaGetLastError(); return ARCHE_ECUDA; }
  memcpy(h_handle64, &h, 64);
  return ARCHE_OK;
}
extern "C" int arche_ipc_open(const unsigned char *h_handle64, void **d_out) {
  if (!h_handle64 || !d_out) return ARCHE_EINVAL;
  cudaIpcMemHandle_t h;
  memcpy(&h, h_handle64, 64);
  *d_out = nullptr;
  if (cudaIpcOpenMemHandle(d_out, h, cudaIpcMemLazyEnablePeerAccess) != cudaSuccess) { (void)cudaGetLastError(); return ARCHE_ECUDA; }
  return ARCHE_OK;
}
extern "C" int arche_ipc_close(void *d_ptr) { return cudaIpcCloseMemHandle(d_ptr) == cudaSuccess ? ARCHE_OK : ARCHE_ECUDA; }

// arche_fft3d without caller scratch and without any allocation: the intermediate passes go through the file-scope
// device array (see its declaration above).  Nothing in it has to start at zero: the first pass writes all Nx*Ny*Nz
// elements before any later pass reads them.  All calls on a device share the array.
extern "C" int arche_fft3d_static(arche_ctx *c, const double *d_in, double *d_out, int sign) {
  if (!c || !d_in || !d_out || (sign != 1 && sign != -1)) return ARCHE_EINVAL;
  if (c->ng > (long long)ARCHE_FFT3D_STATIC_MAX_POINTS) {
    snprintf(c->err, sizeof(c->err), "arche_fft3d_static: grid of %lld points exceeds ARCHE_FFT3D_STATIC_MAX_POINTS = %d "
             "(use arche_fft3d with caller scratch)", c->ng, (int)ARCHE_FFT3D_STATIC_MAX_POINTS);
    return ARCHE_EINVAL;
  }
  if (!c->fft_static) return fail(c, ARCHE_ECUDA, "static FFT scratch address was not taken at set-up");
  return arche_fft3d(c, d_in, d_out, reinterpret_cast<double *>(c->fft_static), sign);
}

extern "C" int arche_rfft3d_forward(arche_ctx *c, const double *d_real_in, double *d_full_out) {
  if (!c || !d_real_in || !d_full_out) return ARCHE_EINVAL;
  int rc = fft3d_forward(c, LoadReal{d_real_in}, StoreComplex{c->work});
  if (rc) return rc;
  expand_half_kernel<<<c->ew_grid, 256, 0, c->stream>>>((double2 *)d_full_out, c->work, c->work, nullptr, c->G.nx, c->G.ny, c->G.nz, c->P);
  LAUNCHED(c);
  return ARCHE_OK;
}

extern "C" int arche_rfft3d_inverse(arche_ctx *c, const double *d_full_in, double *d_real_out) {
  if (!c || !d_full_in || !d_real_out) return ARCHE_EINVAL;
  compress_half_kernel<<<c->ew_grid, 256, 0, c->stream>>>(c->work, (const double2 *)d_full_in, c->G.nx, c->G.ny, c->G.nz, c->P);
  LAUNCHED(c);
  return fft3d_inverse(c, LoadComplex{c->work}, StoreRealPlain{d_real_out});
}

extern "C" int arche_fermi_dirac(arche_ctx *c, int twice_j, const double *d_eta, double *d_out, size_t n) {
  if (!c || !d_eta || !d_out || (twice_j != -1 && twice_j != 1 && twice_j != 3)) return ARCHE_EINVAL;
  if (n == 0) return ARCHE_OK;
  int blocks = (int)((n + 255) / 256 < (size_t)kEwBlocks ? (n + 255) / 256 : kEwBlocks);
  fermi_dirac_kernel<<<blocks, 256, kFdTabBytes, c->stream>>>(twice_j, d_eta, d_out, n, c->fdtab);
  LAUNCHED(c);
  return ARCHE_OK;
}

extern "C" int arche_set_scf_iterations(arche_ctx *c, int scf_max_iter, int scf_fixed_iter) {
  if (!c || scf_max_iter < 0 || scf_fixed_iter < 0) return ARCHE_EINVAL;
  if (scf_max_iter > 0) c->p.scf_max_iter = scf_max_iter;
  c->p.scf_fixed_iter = scf_fixed_iter;
  return ARCHE_OK;
}

extern "C" int arche_is_fused(const arche_ctx *c) { return c && c->fuse ? 1 : 0; }

extern "C" int arche_is_persistent(const arche_ctx *c) {
  if (!c || !c->persist) return 0;
  const int nx = c->G.nx, ny = c->G.ny, nz = c->G.nz;
  return (nx == ny && ny == nz && (nx == 32 || nx == 64)) ? 1 : 0;
}

extern "C" int arche_profile_enable(arche_ctx *c, int on) {
  if (!c) return ARCHE_EINVAL;
  if (on && !c->prof_ev[0])
    for (int k = 0; k < 2 * kProfPairs; ++k) CK(cudaEventCreate(&c->prof_ev[k]));
  CK(cudaStreamSynchronize(c->stream));
  prof_harvest(c);
  c->prof = on != 0;
  if (on) { memset(c->prof_ms, 0, sizeof(c->prof_ms)); memset(c->prof_cnt, 0, sizeof(c->prof_cnt)); }
  return ARCHE_OK;
}

extern "C" int arche_profile_get(arche_ctx *c, int cls, double *h_ms_total, long long *h_launches) {
  if (!c || cls < 0 || cls >= kProfClasses || !h_ms_total || !h_launches) return ARCHE_EINVAL;
  CK(cudaStreamSynchronize(c->stream));
  prof_harvest(c);
  *h_ms_total = c->prof_ms[cls]; *h_launches = c->prof_cnt[cls];
  return ARCHE_OK;
}

// ---- measured rooflines (peak_kernels.cuh) -----------------------------------------------------------------
extern "C" int arche_peak_fp64(arche_ctx *c, double seconds, double *h_tflops, double *h_ms) {
  if (!c || !h_tflops || !(seconds > 0.0)) return ARCHE_EINVAL;
  cudaEvent_t e0, e1;
  CK(cudaEventCreate(&e0)); CK(cudaEventCreate(&e1));
  const int blocks = c->sm_count * 8;
  const long long iters = 200000;                      // ~25 ms per launch at the nominal rate
  double *out = c->partials;                           // never written (see the kernel)
  for (int w = 0; w < 2; ++w) { fp64_fma_peak_kernel<<<blocks, 256, 0, c->stream>>>(iters, 0.999999, 1e-6, out); LAUNCHED(c); }
  double total_ms = 0.0, best_ms = 1e300; long long n = 0;
  while (total_ms < 1e3 * seconds && n < 4096) {
    CK(cudaEventRecord(e0, c->stream));
    fp64_fma_peak_kernel<<<blocks, 256, 0, c->stream>>>(iters, 0.999999, 1e-6, out); LAUNCHED(c);
    CK(cudaEventRecord(e1, c->stream));
    CK(cudaEventSynchronize(e1));
    float ms = 0.f; CK(cudaEventElapsedTime(&ms, e0, e1));
    total_ms += ms; ++n; if (ms < best_ms) best_ms = ms;
  }
  const double flops = 2.0 * (double)kPeakChains * (double)iters * 256.0 * (double)blocks;
  h_tflops[0] = flops * (double)n / (total_ms * 1e-3) / 1e12;   // sustained over the whole run
  h_tflops[1] = flops / (best_ms * 1e-3) / 1e12;                 // best single launch
  if (h_ms) *h_ms = total_ms;
  cudaEventDestroy(e0); cudaEventDestroy(e1);
  return ARCHE_OK;
}

extern "C" int arche_peak_l2(arche_ctx *c, double *h_gbs) {
  if (!c || !h_gbs) return ARCHE_EINVAL;
  cudaEvent_t e0, e1;
  CK(cudaEventCreate(&e0)); CK(cudaEventCreate(&e1));
  // the leading arrays of the workspace (n_i, n_a, V_i, ...): whatever they hold, at most 32 MiB of them
  const size_t avail = (size_t)((const char *)c->kx - (const char *)c->n_i), want = (size_t)32 << 20;
  const long long n = (long long)((avail < want ? avail : want) / sizeof(double2));
  const int blocks = c->sm_count * 8, reps = 64;
  const double2 *buf = reinterpret_cast<const double2 *>(c->n_i);
  l2_read_peak_kernel<<<blocks, 256, 0, c->stream>>>(buf, n, 4, c->partials); LAUNCHED(c);
  double best = 1e300;
  for (int k = 0; k < 5; ++k) {
    CK(cudaEventRecord(e0, c->stream));
    l2_read_peak_kernel<<<blocks, 256, 0, c->stream>>>(buf, n, reps, c->partials); LAUNCHED(c);
    CK(cudaEventRecord(e1, c->stream));
    CK(cudaEventSynchronize(e1));
    float ms = 0.f; CK(cudaEventElapsedTime(&ms, e0, e1));
    if (ms < best) best = ms;
  }
  *h_gbs = (double)n * sizeof(double2) * reps / (best * 1e-3) / 1e9;
  cudaEventDestroy(e0); cudaEventDestroy(e1);
  return ARCHE_OK;
}
