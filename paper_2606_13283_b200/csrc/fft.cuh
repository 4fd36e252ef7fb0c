// fft.cuh -- hand-written fp64 3D FFT for sm_100a (no cuFFT anywhere on the product path): the GENERIC passes for any
// 2^a 3^b length (shared-memory Stockham stages, run-time radix plan) and the functor protocol.  The production
// sizes 32..384 take the register two-stage passes of fft_fast.cuh; these kernels serve every other length, the
// stand-alone complex transform arche_fft3d, and the r2c / c2r x passes of odd-sized grids.
//
// One kernel launch per axis.  A block owns a tile of L lines of length N of that axis:
//   axis x: L consecutive x-lines (each line contiguous in memory);
//   axis y/z: L consecutive x positions for a fixed z (or y): every global row of the tile is L*16 contiguous
//             bytes, the "transpose" happens in shared memory ([i][l] layout, l fastest => conflict-free).
// Inside the block: Stockham autosort radix-8/4/3/2 stages ping-ponging between two shared-memory buffers
// (split re/im arrays so that every access is an 8-byte word).  Twiddles come from a per-axis table
// exp(-2 pi i a/N) built on the host in long double.
// The inverse transform uses the swap identity IDFT(x) = swap(DFT(swap(x))) (swap = exchange re and im), so only
// forward butterflies exist.  Pointwise work is fused through LoadOp / StoreOp functors applied when a tile
// is first read / last written (G-space Poisson + V_ie assembly, real-part + V_xc epilogue, reductions).
#pragma once
#include "common.cuh"

namespace arche {

constexpr int kFftThreads = 256;
constexpr int kFftMaxStages = 12;

struct FftAxisPlan {
  int n;
  int nstages;
  int radix[kFftMaxStages];
  const double2 *tw;  // device, [n], exp(-2 pi i a / n)
  const int *stop;    // optional device flag: when set and non-zero the pass is skipped (speculative SCF launches)
};

struct FftPass {
  FftAxisPlan plan;
  int nx, ny, nz;
  int L;  // lines per block
};

struct Cplx { double re, im; };

__device__ __forceinline__ void bfly2(Cplx &a, Cplx &b) {
  Cplx t = {a.re - b.re, a.im - b.im};
  a.re += b.re; a.im += b.im;
  b = t;
}
// forward DFT-4 in place, natural order output
__device__ __forceinline__ void dft4(Cplx &v0, Cplx &v1, Cplx &v2, Cplx &v3) {
  Cplx a = {v0.re + v2.re, v0.im + v2.im}, b = {v0.re - v2.re, v0.im - v2.im};
  Cplx c = {v1.re + v3.re, v1.im + v3.im}, d = {v1.re - v3.re, v1.im - v3.im};
  v0 = {a.re + c.re, a.im + c.im};
  v2 = {a.re - c.re, a.im - c.im};
  v1 = {b.re + d.im, b.im - d.re};  // b - i d
  v3 = {b.re - d.im, b.im + d.re};  // b + i d
}
__device__ __forceinline__ void dft3(Cplx &v0, Cplx &v1, Cplx &v2) {
  const double h = 0.86602540378443864676372317075294;  // sqrt(3)/2
  Cplx s = {v1.re + v2.re, v1.im + v2.im}, d = {v1.re - v2.re, v1.im - v2.im};
  Cplx m = {v0.re - 0.5 * s.re, v0.im - 0.5 * s.im};
  v0 = {v0.re + s.re, v0.im + s.im};
  v1 = {m.re + h * d.im, m.im - h * d.re};
  v2 = {m.re - h * d.im, m.im + h * d.re};
}
__device__ __forceinline__ void dft8(Cplx (&v)[8]) {
  const double c = 0.70710678118654752440084436210485;
  dft4(v[0], v[2], v[4], v[6]);
  dft4(v[1], v[3], v[5], v[7]);
  // odd part times W8^t
  Cplx o1 = {c * (v[3].re + v[3].im), c * (v[3].im - v[3].re)};    // * (c, -c)
  Cplx o2 = {v[5].im, -v[5].re};                                   // * (-i)
  Cplx o3 = {c * (v[7].im - v[7].re), -c * (v[7].re + v[7].im)};   // * (-c, -c)
  Cplx e0 = v[0], e1 = v[2], e2 = v[4], e3 = v[6], o0 = v[1];
  v[0] = {e0.re + o0.re, e0.im + o0.im}; v[4] = {e0.re - o0.re, e0.im - o0.im};
  v[1] = {e1.re + o1.re, e1.im + o1.im}; v[5] = {e1.re - o1.re, e1.im - o1.im};
  v[2] = {e2.re + o2.re, e2.im + o2.im}; v[6] = {e2.re - o2.re, e2.im - o2.im};
  v[3] = {e3.re + o3.re, e3.im + o3.im}; v[7] = {e3.re - o3.re, e3.im - o3.im};
}

template <int R, int AXIS>
__device__ __forceinline__ void fft_stage(const double *__restrict__ sre, const double *__restrict__ sim,
                                          double *__restrict__ dre, double *__restrict__ dim, int N, int Ns, int L,
                                          const double2 *__restrict__ tw) {
  const int nb = N / R;
  const int twmul = N / (Ns * R);
  for (int w = threadIdx.x; w < L * nb; w += blockDim.x) {
    int l, j;
    if (AXIS == 0) { j = w % nb; l = w / nb; } else { l = w % L; j = w / L; }
    const int k = j % Ns;
    Cplx v[R];
#pragma unroll
    for (int t = 0; t < R; ++t) {
      const int i = j + t * nb;
      const int a = (AXIS == 0) ? l * N + i : i * L + l;
      v[t].re = sre[a]; v[t].im = sim[a];
    }
    if (Ns > 1) {
#pragma unroll
      for (int t = 1; t < R; ++t) {
        const double2 wv = __ldg(&tw[t * k * twmul]);
        const double re = v[t].re * wv.x - v[t].im * wv.y;
        v[t].im = v[t].re * wv.y + v[t].im * wv.x;
        v[t].re = re;
      }
    }
    if (R == 2) bfly2(v[0], v[1]);
    if (R == 3) dft3(v[0], v[1], v[2]);
    if (R == 4) dft4(v[0], v[1], v[2], v[3]);
    if (R == 8) dft8(reinterpret_cast<Cplx(&)[8]>(v));
    const int j0 = (j - k) * R + k;
#pragma unroll
    for (int t = 0; t < R; ++t) {
      const int i = j0 + t * Ns;
      const int a = (AXIS == 0) ? l * N + i : i * L + l;
      dre[a] = v[t].re; dim[a] = v[t].im;
    }
  }
}

// Plain complex array load / store functors.
// Functor protocol (all passes): begin() once per thread at kernel start; load: operator()(idx, ix, iy, iz, re, im)
// (complex) or load_real(idx, ix, iy, iz); store(idx, ix, iy, iz, re, im) or store_real(idx, ix, iy, iz, v);
// finish(smem) once per block at the end (grid reductions; smem = the tile buffer, free by then);
// prefetch(idx): L2 prefetch of the operand lines the functor will touch at element idx (fast passes only).
struct LoadComplex {
  static constexpr bool kWriteBack = false;
  const double2 *src;
  __device__ __forceinline__ void begin() {}
  __device__ __forceinline__ void prefetch(long long idx) const { prefetch_l2(src + idx); }
  __device__ __forceinline__ void operator()(long long idx, int, int, int, double &re, double &im) {
    double2 v = src[idx]; re = v.x; im = v.y;
  }
  __device__ __forceinline__ void finish(double *) {}
};
struct StoreComplex {
  static constexpr bool kSplitStore = false;
  double2 *dst;
  __device__ __forceinline__ void begin() {}
  __device__ __forceinline__ void prefetch(long long) const {}
  __device__ __forceinline__ void store(long long idx, int, int, int, double re, double im) { dst[idx] = make_double2(re, im); }
  __device__ __forceinline__ void finish(double *) {}
};

// f4: slab-decomposed transform over several GPUs.  The pass that precedes the transpose stores every
// element straight into the slab of the rank that owns it after the transpose -- peer memory mapped over NVLink (or,
// with one rank, the local buffer): the all-to-all is the store phase of the pass, there is no pack/exchange/unpack.
// Forward: the y pass of rank r, working on its z slab [nzl][ny][nx], writes (ix, iy, izl) to rank q = iy / nyl at
// [(r nzl + izl)][iy - q nyl][ix] of that rank's y slab [nz][nyl][nx].  Inverse: the z pass of rank r, working on its y
// slab, writes (ix, iyl, iz) to rank q = iz / nzl at [iz - q nzl][r nyl + iyl][ix] of that rank's z slab.
constexpr int kSlabMaxRanks = 16;
struct StoreSlabScatter {
  static constexpr bool kSplitStore = false;
  double2 *peer[kSlabMaxRanks];
  int nx, nloc_dst;     // row length; slab thickness of the destination layout (nyl forward, nzl inverse)
  int pitch_dst;        // middle extent of the destination layout (nyl forward, ny inverse)
  int off_src;          // this rank's offset along the axis it owned before the transpose (r nzl forward, r nyl inverse)
  int forward;
  __device__ __forceinline__ void begin() {}
  __device__ __forceinline__ void prefetch(long long) const {}
  __device__ __forceinline__ void store(long long, int ix, int iy, int iz, double re, double im) {
    if (forward) {
      const int q = iy / nloc_dst;
      peer[q][((long long)(off_src + iz) * pitch_dst + (iy - q * nloc_dst)) * nx + ix] = make_double2(re, im);
    } else {
      const int q = iz / nloc_dst;
      peer[q][((long long)(iz - q * nloc_dst) * pitch_dst + (off_src + iy)) * nx + ix] = make_double2(re, im);
    }
  }
  __device__ __forceinline__ void finish(double *) {}
};

template <int AXIS, bool INVERSE, class LoadOp, class StoreOp>
__global__ void __launch_bounds__(kFftThreads) fft_pass_kernel(FftPass P, LoadOp ld_in, StoreOp st_in) {
  extern __shared__ double smem[];
  const int N = P.plan.n, L = P.L;
  double *b0re = smem, *b0im = smem + (size_t)L * N, *b1re = smem + 2 * (size_t)L * N, *b1im = smem + 3 * (size_t)L * N;
  StoreOp st = st_in;
  LoadOp ld = ld_in;
  if (P.plan.stop && *P.plan.stop) return;
  ld.begin(); st.begin();
  // tile geometry
  const long long nxny = (long long)P.nx * P.ny;
  long long tile_base;
  int fx = 0, fy = 0, fz = 0;  // fixed coordinates of the tile origin
  if (AXIS == 0) {
    long long line0 = (long long)blockIdx.x * L;  // line = iy + ny*iz
    tile_base = line0 * P.nx;
    fy = (int)(line0 % P.ny); fz = (int)(line0 / P.ny);
  } else if (AXIS == 1) {
    const int xt = P.nx / L;
    fz = blockIdx.x / xt; fx = (blockIdx.x % xt) * L;
    tile_base = fz * nxny + fx;
  } else {
    const int xt = P.nx / L;
    fy = blockIdx.x / xt; fx = (blockIdx.x % xt) * L;
    tile_base = (long long)fy * P.nx + fx;
  }
  const long long estride = AXIS == 0 ? 1 : (AXIS == 1 ? P.nx : nxny);
  // ---- load tile
  for (int e = threadIdx.x; e < L * N; e += blockDim.x) {
    int l, i;
    if (AXIS == 0) { i = e % N; l = e / N; } else { l = e % L; i = e / L; }
    long long idx; int ix, iy, iz;
    if (AXIS == 0) {
      idx = tile_base + (long long)l * N + i;
      ix = i; int ln = fy + l; iy = ln % P.ny; iz = fz + ln / P.ny;
    } else if (AXIS == 1) {
      idx = tile_base + i * estride + l; ix = fx + l; iy = i; iz = fz;
    } else {
      idx = tile_base + i * estride + l; ix = fx + l; iy = fy; iz = i;
    }
    double re, im;
    ld(idx, ix, iy, iz, re, im);
    const int a = (AXIS == 0) ? l * N + i : i * L + l;
    if (INVERSE) { b0re[a] = im; b0im[a] = re; } else { b0re[a] = re; b0im[a] = im; }
  }
  __syncthreads();
  // ---- Stockham stages
  double *sre = b0re, *sim = b0im, *dre = b1re, *dim = b1im;
  int Ns = 1;
  for (int s = 0; s < P.plan.nstages; ++s) {
    const int R = P.plan.radix[s];
    if (R == 8) fft_stage<8, AXIS>(sre, sim, dre, dim, N, Ns, L, P.plan.tw);
    else if (R == 4) fft_stage<4, AXIS>(sre, sim, dre, dim, N, Ns, L, P.plan.tw);
    else if (R == 3) fft_stage<3, AXIS>(sre, sim, dre, dim, N, Ns, L, P.plan.tw);
    else fft_stage<2, AXIS>(sre, sim, dre, dim, N, Ns, L, P.plan.tw);
    __syncthreads();
    double *t;
    t = sre; sre = dre; dre = t;
    t = sim; sim = dim; dim = t;
    Ns *= R;
  }
  // ---- store tile
  for (int e = threadIdx.x; e < L * N; e += blockDim.x) {
    int l, i;
    if (AXIS == 0) { i = e % N; l = e / N; } else { l = e % L; i = e / L; }
    long long idx; int ix, iy, iz;
    if (AXIS == 0) {
      idx = tile_base + (long long)l * N + i;
      ix = i; int ln = fy + l; iy = ln % P.ny; iz = fz + ln / P.ny;
    } else if (AXIS == 1) {
      idx = tile_base + i * estride + l; ix = fx + l; iy = i; iz = fz;
    } else {
      idx = tile_base + i * estride + l; ix = fx + l; iy = fy; iz = i;
    }
    const int a = (AXIS == 0) ? l * N + i : i * L + l;
    if (INVERSE) st.store(idx, ix, iy, iz, sim[a], sre[a]); else st.store(idx, ix, iy, iz, sre[a], sim[a]);
  }
  __syncthreads();
  ld.finish(smem);
  st.finish(smem);
}

// ---- x passes on real data (half spectrum) ---------------------------------------------------------
// The real field [nz][ny][nx] transforms to the half spectrum [nz][ny][P] (ix = 0..nx/2 stored, row pitch P >= nx/2+1,
// columns ix >= nx/2+1 are zero padding).  Two real lines a, b are packed as z = a + i b, one complex FFT of
// length nx gives Z, and A(k) = (Z(k) + conj Z(N-k))/2, B(k) = (Z(k) - conj Z(N-k))/(2i) are the two half spectra.
// The inverse builds Z = A + i B (completed by Hermitian symmetry) and one complex inverse FFT returns a = Re z,
// b = Im z.  A block owns LP line pairs; stages run in shared memory ([pair][i] layout).
struct FftRealPass {
  FftAxisPlan plan;
  int nx, ny, nz;
  int P;    // row pitch of the half spectrum (complex elements)
  int LP;   // line pairs per block
};

__device__ __forceinline__ void fft_run_stages_x(const FftAxisPlan &plan, int LP, double *&sre, double *&sim, double *&dre,
                                                 double *&dim) {
  const int N = plan.n;
  int Ns = 1;
  for (int s = 0; s < plan.nstages; ++s) {
    const int R = plan.radix[s];
    if (R == 8) fft_stage<8, 0>(sre, sim, dre, dim, N, Ns, LP, plan.tw);
    else if (R == 4) fft_stage<4, 0>(sre, sim, dre, dim, N, Ns, LP, plan.tw);
    else if (R == 3) fft_stage<3, 0>(sre, sim, dre, dim, N, Ns, LP, plan.tw);
    else fft_stage<2, 0>(sre, sim, dre, dim, N, Ns, LP, plan.tw);
    __syncthreads();
    double *t;
    t = sre; sre = dre; dre = t;
    t = sim; sim = dim; dim = t;
    Ns *= R;
  }
}

// forward: real lines -> half spectrum.  LoadOp: double load_real(idx, ix, iy, iz); StoreOp: store(idx, ix, iy, iz, re, im)
template <class LoadOp, class StoreOp>
__global__ void __launch_bounds__(kFftThreads) fft_r2c_x_kernel(FftRealPass P, LoadOp ld_in, StoreOp st_in) {
  extern __shared__ double smem[];
  const int N = P.plan.n, LP = P.LP, nxh = N / 2 + 1;
  double *sre = smem, *sim = smem + (size_t)LP * N, *dre = smem + 2 * (size_t)LP * N, *dim = smem + 3 * (size_t)LP * N;
  LoadOp ld = ld_in;
  StoreOp st = st_in;
  if (P.plan.stop && *P.plan.stop) return;
  ld.begin(); st.begin();
  const long long nl = (long long)P.ny * P.nz;
  const long long line_base = (long long)blockIdx.x * LP * 2;
  for (int e = threadIdx.x; e < 2 * LP * N; e += blockDim.x) {  // consecutive lines, contiguous in memory
    const int i = e % N, q = e / N;                              // q = line within the tile (pair q/2, member q%2)
    const long long line = line_base + q;
    double v = 0.0;
    if (line < nl) v = ld.load_real(line * N + i, i, (int)(line % P.ny), (int)(line / P.ny));
    if (q & 1) sim[(q >> 1) * N + i] = v; else sre[(q >> 1) * N + i] = v;
  }
  __syncthreads();
  fft_run_stages_x(P.plan, LP, sre, sim, dre, dim);
  for (int e = threadIdx.x; e < 2 * LP * P.P; e += blockDim.x) {
    const int k = e % P.P, q = e / P.P, pr = q >> 1;
    const long long line = line_base + q;
    if (line >= nl) continue;
    double re = 0.0, im = 0.0;
    if (k < nxh) {
      const int mk = k == 0 ? 0 : N - k;
      const double zr = sre[pr * N + k], zi = sim[pr * N + k], mr = sre[pr * N + mk], mi = sim[pr * N + mk];
      if (q & 1) { re = 0.5 * (zi + mi); im = -0.5 * (zr - mr); }   // B(k)
      else { re = 0.5 * (zr + mr); im = 0.5 * (zi - mi); }          // A(k)
    }
    st.store(line * P.P + k, k, (int)(line % P.ny), (int)(line / P.ny), re, im);
  }
  __syncthreads();
  ld.finish(smem);
  st.finish(smem);
}

// inverse: half spectrum -> real lines (unnormalised).  LoadOp: operator()(idx, ix, iy, iz, re, im);
// StoreOp: store_real(idx, ix, iy, iz, v)
template <class LoadOp, class StoreOp>
__global__ void __launch_bounds__(kFftThreads) fft_c2r_x_kernel(FftRealPass P, LoadOp ld_in, StoreOp st_in) {
  extern __shared__ double smem[];
  const int N = P.plan.n, LP = P.LP, nxh = N / 2 + 1;
  double *sre = smem, *sim = smem + (size_t)LP * N, *dre = smem + 2 * (size_t)LP * N, *dim = smem + 3 * (size_t)LP * N;
  LoadOp ld = ld_in;
  StoreOp st = st_in;
  if (P.plan.stop && *P.plan.stop) return;
  ld.begin(); st.begin();
  const long long nl = (long long)P.ny * P.nz;
  const long long line_base = (long long)blockIdx.x * LP * 2;
  for (int e = threadIdx.x; e < LP * nxh; e += blockDim.x) {
    const int k = e % nxh, pr = e / nxh;
    const long long la = line_base + 2 * pr, lb = la + 1;
    double ar = 0.0, ai = 0.0, br = 0.0, bi = 0.0;
    if (la < nl) ld(la * P.P + k, k, (int)(la % P.ny), (int)(la / P.ny), ar, ai);
    if (lb < nl) ld(lb * P.P + k, k, (int)(lb % P.ny), (int)(lb / P.ny), br, bi);
    // conj(Z(k)), Z = A + i B  (inverse transform = conj . forward . conj)
    sre[pr * N + k] = ar - bi; sim[pr * N + k] = -(ai + br);
    const int mk = N - k;
    if (k > 0 && mk >= nxh) { sre[pr * N + mk] = ar + bi; sim[pr * N + mk] = ai - br; }  // conj(conj A + i conj B)
  }
  __syncthreads();
  fft_run_stages_x(P.plan, LP, sre, sim, dre, dim);
  for (int e = threadIdx.x; e < 2 * LP * N; e += blockDim.x) {
    const int i = e % N, q = e / N;
    const long long line = line_base + q;
    if (line >= nl) continue;
    const double v = (q & 1) ? -sim[(q >> 1) * N + i] : sre[(q >> 1) * N + i];
    st.store_real(line * N + i, i, (int)(line % P.ny), (int)(line / P.ny), v);
  }
  __syncthreads();
  ld.finish(smem);
  st.finish(smem);
}

// ---- host side ------------------------------------------------------------------------------
static inline bool fft_make_plan(int n, const double2 *d_tw, FftAxisPlan *p) {
  p->n = n; p->tw = d_tw; p->nstages = 0; p->stop = nullptr;
  int m = n;
  // radix-3 factors first (small Ns => no twiddles on the odd radix), then 8s, then the 4/2 remainder
  while (m % 3 == 0) { p->radix[p->nstages++] = 3; m /= 3; }
  while (m % 8 == 0) { p->radix[p->nstages++] = 8; m /= 8; }
  if (m % 4 == 0) { p->radix[p->nstages++] = 4; m /= 4; }
  if (m % 2 == 0) { p->radix[p->nstages++] = 2; m /= 2; }
  return m == 1 && p->nstages <= kFftMaxStages;
}

static inline int fft_pick_L(int axis, int n, int nx, int ny, int nz) {
  const int max_elems = 3072;  // 4 arrays * 8 B * L*N <= 96 KB
  if (axis == 0) {
    long long lines = (long long)ny * nz;
    int L = 1;
    while (L * 2 * n <= max_elems && lines % (L * 2) == 0 && L < 64) L *= 2;
    return L;
  }
  int L = 1;
  while (L * 2 * n <= max_elems && nx % (L * 2) == 0 && L < 16) L *= 2;
  return L;
}

template <int AXIS, bool INVERSE, class LoadOp, class StoreOp>
static inline cudaError_t fft_launch_pass(const FftAxisPlan &plan, int nx, int ny, int nz, LoadOp ld, StoreOp st,
                                          cudaStream_t stream, int *blocks_out = nullptr) {
  FftPass P;
  P.plan = plan; P.nx = nx; P.ny = ny; P.nz = nz;
  P.L = fft_pick_L(AXIS, plan.n, nx, ny, nz);
  long long blocks = AXIS == 0 ? (long long)ny * nz / P.L : (AXIS == 1 ? (long long)nz * (nx / P.L) : (long long)ny * (nx / P.L));
  size_t smem = 4 * sizeof(double) * (size_t)P.L * plan.n;
  if (smem < 4096) smem = 4096;  // room for the reduction scratch used by finish()
  auto kern = fft_pass_kernel<AXIS, INVERSE, LoadOp, StoreOp>;
  static int attr_dev = -1;   // the opt-in is per device
  int dev = 0;
  cudaGetDevice(&dev);
  if (attr_dev != dev) {
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, 100 * 1024);
    if (e != cudaSuccess) return e;
    attr_dev = dev;
  }
  if (blocks_out) *blocks_out = (int)blocks;
  kern<<<(unsigned)blocks, kFftThreads, smem, stream>>>(P, ld, st);
  return cudaGetLastError();
}

static inline int fft_pick_LP(int n, long long lines) {
  const int max_elems = 3072;  // 4 arrays * 8 B * LP*N <= 96 KB
  const long long pairs = (lines + 1) / 2;
  int LP = 1;
  while (LP * 2 * n <= max_elems && LP * 2 <= pairs && LP < 32) LP *= 2;
  return LP;
}
static inline int fft_real_blocks(int n, int ny, int nz) {
  const long long lines = (long long)ny * nz, pairs = (lines + 1) / 2;
  const int LP = fft_pick_LP(n, lines);
  return (int)((pairs + LP - 1) / LP);
}

template <bool INVERSE, class LoadOp, class StoreOp>
static inline cudaError_t fft_launch_real_x(const FftAxisPlan &plan, int nx, int ny, int nz, int pitch, LoadOp ld, StoreOp st,
                                            cudaStream_t stream) {
  FftRealPass P;
  P.plan = plan; P.nx = nx; P.ny = ny; P.nz = nz; P.P = pitch;
  P.LP = fft_pick_LP(nx, (long long)ny * nz);
  const int blocks = fft_real_blocks(nx, ny, nz);
  size_t smem = 4 * sizeof(double) * (size_t)P.LP * plan.n;
  if (smem < 4096) smem = 4096;
  static int attr_dev = -1;
  int dev = 0;
  cudaGetDevice(&dev);
  const bool attr_set = attr_dev == dev;
  if constexpr (INVERSE) {
    auto kern = fft_c2r_x_kernel<LoadOp, StoreOp>;
    if (!attr_set) {
      cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, 100 * 1024);
      if (e != cudaSuccess) return e;
      attr_dev = dev;
    }
    kern<<<blocks, kFftThreads, smem, stream>>>(P, ld, st);
  } else {
    auto kern = fft_r2c_x_kernel<LoadOp, StoreOp>;
    if (!attr_set) {
      cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, 100 * 1024);
      if (e != cudaSuccess) return e;
      attr_dev = dev;
    }
    kern<<<blocks, kFftThreads, smem, stream>>>(P, ld, st);
  }
  return cudaGetLastError();
}

}  // namespace arche
