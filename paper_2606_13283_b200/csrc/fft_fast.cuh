// fft_fast.cuh -- two-stage register FFT passes for the production grid sizes (N = R1*R2 in {32, 64, 128, 192, 256, 384}).
//
// Every thread holds one radix-R butterfly (R up to 24) in registers; a 1D transform of length N = R1*R2 is
//   stage 1:  y[j1*R1 + t'] = DFT_R1{ x[j1 + t*R2] }_t                      j1 in [0,R2)     (no twiddles)
//   stage 2:  X[j2 + t'*R1] = DFT_R2{ W_N^(t*j2) y[j2 + t*R1] }_t            j2 in [0,R1)
// with exactly one exchange through shared memory between the stages (Stockham autosort, natural order in and out).
//   y/z passes: a block owns 8 consecutive x columns (128-byte rows) and all N points of the axis; stage 1 reads global
//               memory straight into registers, stage 2 stores straight from registers (one smem round trip in total).
//   x passes:   real <-> half-spectrum (see fft.cuh): a block owns LP pairs of contiguous real lines; the pointwise
//               prologue/epilogue functors run on all threads, two lines of a pair per thread (one 16-byte smem word).
// The inverse transform is conj . forward . conj.  Butterflies larger than 4 are Cooley-Tukey compositions in
// registers with compile-time twiddles (table of cos(2 pi k/48)).
#pragma once
#include <type_traits>

#include "fft.cuh"

namespace arche {

// ---- compile-time twiddles -------------------------------------------------------------------------------
__host__ __device__ constexpr double cos48_quarter(int k) {  // cos(2 pi k/48), k = 0..12
  constexpr double t[13] = {1.0, 0.99144486137381041114, 0.96592582628906828675, 0.92387953251128675613,
                            0.86602540378443864676, 0.79335334029123516458, 0.7071067811865475244,
                            0.60876142900872063942, 0.5, 0.38268343236508977173, 0.25881904510252076235,
                            0.13052619222005159155, 0.0};
  return t[k];
}
__host__ __device__ constexpr double cos48(int k) {
  k = ((k % 48) + 48) % 48;
  if (k > 24) k = 48 - k;
  return k > 12 ? -cos48_quarter(24 - k) : cos48_quarter(k);
}
__host__ __device__ constexpr double sin48(int k) { return cos48(k + 36); }  // sin(t) = cos(t - 90 deg)

__device__ __forceinline__ double2 cadd(double2 a, double2 b) { return make_double2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ double2 csub(double2 a, double2 b) { return make_double2(a.x - b.x, a.y - b.y); }
__device__ __forceinline__ double2 cmul(double2 a, double2 b) {
  return make_double2(fma(a.x, b.x, -a.y * b.y), fma(a.x, b.y, a.y * b.x));
}

// v * exp(-2 pi i NUM/DEN), DEN | 48
template <int NUM, int DEN>
__device__ __forceinline__ double2 twid(double2 v) {
  constexpr int k = ((NUM % DEN) + DEN) % DEN * (48 / DEN);  // angle = 2 pi k/48
  if constexpr (k == 0) return v;
  else if constexpr (k == 12) return make_double2(v.y, -v.x);   // * (-i)
  else if constexpr (k == 24) return make_double2(-v.x, -v.y);
  else if constexpr (k == 36) return make_double2(-v.y, v.x);   // * (+i)
  else if constexpr (k == 6) { constexpr double c = cos48(6); return make_double2(c * (v.x + v.y), c * (v.y - v.x)); }
  else if constexpr (k == 18) { constexpr double c = cos48(6); return make_double2(c * (v.y - v.x), -c * (v.x + v.y)); }
  else if constexpr (k == 30) { constexpr double c = cos48(6); return make_double2(-c * (v.x + v.y), c * (v.x - v.y)); }
  else if constexpr (k == 42) { constexpr double c = cos48(6); return make_double2(c * (v.x - v.y), c * (v.x + v.y)); }
  else { constexpr double c = cos48(k), s = sin48(k); return make_double2(fma(v.x, c, v.y * s), fma(v.y, c, -v.x * s)); }
}

// ---- in-register DFTs (forward, natural order in and out) ------------------------------------------------
template <int R> struct Dft;
template <> struct Dft<2> {
  static __device__ __forceinline__ void run(double2 (&v)[2]) { const double2 a = v[0]; v[0] = cadd(a, v[1]); v[1] = csub(a, v[1]); }
};
template <> struct Dft<3> {
  static __device__ __forceinline__ void run(double2 (&v)[3]) {
    constexpr double h = 0.86602540378443864676;
    const double2 s = cadd(v[1], v[2]), d = csub(v[1], v[2]);
    const double2 m = make_double2(v[0].x - 0.5 * s.x, v[0].y - 0.5 * s.y);
    v[0] = cadd(v[0], s);
    v[1] = make_double2(m.x + h * d.y, m.y - h * d.x);
    v[2] = make_double2(m.x - h * d.y, m.y + h * d.x);
  }
};
template <> struct Dft<4> {
  static __device__ __forceinline__ void run(double2 (&v)[4]) {
    const double2 a = cadd(v[0], v[2]), b = csub(v[0], v[2]), c = cadd(v[1], v[3]), d = csub(v[1], v[3]);
    v[0] = cadd(a, c); v[2] = csub(a, c);
    v[1] = make_double2(b.x + d.y, b.y - d.x);   // b - i d
    v[3] = make_double2(b.x - d.y, b.y + d.x);   // b + i d
  }
};
template <int I, int N, class F>
__device__ __forceinline__ void static_for(F &&f) {
  if constexpr (I < N) { f(std::integral_constant<int, I>{}); static_for<I + 1, N>(f); }
}
// R = A*B (n = A n2 + n1, k = B k1 + k2): DFT_B over the stride-A subsequences, twiddle W_R^(n1 k2), DFT_A over the
// contiguous groups, transpose to natural order
template <int A, int B>
__device__ __forceinline__ void dft_ct(double2 (&v)[A * B]) {
  constexpr int R = A * B;
  static_for<0, A>([&](auto n1c) {
    constexpr int n1 = decltype(n1c)::value;
    double2 t[B];
    static_for<0, B>([&](auto n2c) { constexpr int n2 = decltype(n2c)::value; t[n2] = v[A * n2 + n1]; });
    Dft<B>::run(t);
    static_for<0, B>([&](auto k2c) { constexpr int k2 = decltype(k2c)::value; v[A * k2 + n1] = twid<n1 * k2, R>(t[k2]); });
  });
  double2 o[R];
  static_for<0, B>([&](auto k2c) {
    constexpr int k2 = decltype(k2c)::value;
    double2 t[A];
    static_for<0, A>([&](auto n1c) { constexpr int n1 = decltype(n1c)::value; t[n1] = v[A * k2 + n1]; });
    Dft<A>::run(t);
    static_for<0, A>([&](auto k1c) { constexpr int k1 = decltype(k1c)::value; o[B * k1 + k2] = t[k1]; });
  });
  static_for<0, R>([&](auto ic) { constexpr int i = decltype(ic)::value; v[i] = o[i]; });
}
template <> struct Dft<6> { static __device__ __forceinline__ void run(double2 (&v)[6]) { dft_ct<2, 3>(v); } };
template <> struct Dft<8> { static __device__ __forceinline__ void run(double2 (&v)[8]) { dft_ct<2, 4>(v); } };
template <> struct Dft<12> { static __device__ __forceinline__ void run(double2 (&v)[12]) { dft_ct<3, 4>(v); } };
template <> struct Dft<16> { static __device__ __forceinline__ void run(double2 (&v)[16]) { dft_ct<4, 4>(v); } };
template <> struct Dft<24> { static __device__ __forceinline__ void run(double2 (&v)[24]) { dft_ct<3, 8>(v); } };

// ---- plans -----------------------------------------------------------------------------------------------
template <int N> struct FastPlan { static constexpr bool ok = false; static constexpr int R1 = 1, R2 = 1; };
template <> struct FastPlan<32> { static constexpr bool ok = true; static constexpr int R1 = 4, R2 = 8; };
template <> struct FastPlan<64> { static constexpr bool ok = true; static constexpr int R1 = 8, R2 = 8; };
template <> struct FastPlan<128> { static constexpr bool ok = true; static constexpr int R1 = 8, R2 = 16; };
template <> struct FastPlan<192> { static constexpr bool ok = true; static constexpr int R1 = 12, R2 = 16; };
template <> struct FastPlan<256> { static constexpr bool ok = true; static constexpr int R1 = 16, R2 = 16; };
template <> struct FastPlan<384> { static constexpr bool ok = true; static constexpr int R1 = 16, R2 = 24; };

struct LoadReal;   // scf_kernels.cuh: plain real input (the one load functor the copy-engine r2c pass replaces)
struct FastGeom {
  int nx, ny, nz, P;        // real grid and half-spectrum pitch
  const double2 *tw;        // exp(-2 pi i a/N) of the transformed axis
  const int *stop;          // optional device flag: non-zero skips the pass
  int pdl;                  // host side: launch with programmatic stream serialization (common.cuh)
  int tma;                  // host side: plain r2c x pass with its input through the copy engine (fft_r2c_tma_kernel)
};

// kernel launch with optional programmatic dependent launch
static inline cudaError_t launch_maybe_pdl(const void *kern, dim3 grid, dim3 block, void **args, size_t smem, cudaStream_t stream, bool pdl) {
  if (!pdl) return cudaLaunchKernel(kern, grid, block, args, smem, stream);
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = stream;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = at; cfg.numAttrs = 1;
  return cudaLaunchKernelExC(&cfg, kern, args);
}

constexpr int kFastL = 8;   // columns per y/z tile (128-byte rows)
template <int N> __host__ __device__ constexpr int fast_threads_yz() {
  return kFastL * (FastPlan<N>::R1 > FastPlan<N>::R2 ? FastPlan<N>::R1 : FastPlan<N>::R2);
}

// barrier over a group of `count` threads (multiple of 32) of the block; id 0 with the whole block = __syncthreads()
__device__ __forceinline__ void group_sync(int id, int count) { asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(count) : "memory"); }

// ---- y / z pass over the half spectrum [nz][ny][P] -------------------------------------------------------
// One tile (8 columns x N) by a group of fast_threads_yz<N>() threads: t = thread index within the group, buf = the
// group's [N][8] shared buffer, bar = the group's barrier id.  Used by the per-pass kernel (group = block) and by the
// persistent SCF kernel (several groups per block).
template <int N, int AXIS, bool INVERSE, bool PREFETCH, class LoadOp, class StoreOp>
__device__ __forceinline__ void fft_yz_tile(const FastGeom &G, LoadOp &ld, StoreOp &st, int tile, double2 *buf, int t_in_group,
                                            int bar) {
  constexpr int R1 = FastPlan<N>::R1, R2 = FastPlan<N>::R2, TH = fast_threads_yz<N>(), JS = TH / kFastL;
  const int l = t_in_group % kFastL, jj = t_in_group / kFastL;
  const int xt = G.P / kFastL;
  const int fixed = tile / xt, ix = (tile % xt) * kFastL + l;   // fixed = iz (AXIS 1) or iy (AXIS 2)
  const long long stride = AXIS == 1 ? G.P : (long long)G.P * G.ny;
  const long long base = (AXIS == 1 ? (long long)fixed * G.ny * G.P : (long long)fixed * G.P) + ix;
  if (PREFETCH && l == 0) {  // one lane per 128-byte row: request every operand line of the tile now
    for (int j1 = jj; j1 < R2; j1 += JS)
#pragma unroll
      for (int t = 0; t < R1; ++t) ld.prefetch(base + (j1 + t * R2) * stride);
    for (int j2 = jj; j2 < R1; j2 += JS)
#pragma unroll
      for (int t = 0; t < R2; ++t) st.prefetch(base + (j2 + t * R1) * stride);
  }
  // stage 1: global -> registers -> shared
  for (int j1 = jj; j1 < R2; j1 += JS) {
    double2 v[R1];
    if constexpr (LoadOp::kWriteBack && R1 <= 8) {
      // a prologue that also updates its operand in place: all loads first, then the stores, so that the stores
      // (which the compiler must assume to alias the next loads) do not serialise the load latencies
      double2 wb[R1];
#pragma unroll
      for (int t = 0; t < R1; ++t) {
        const int i = j1 + t * R2;
        ld.load_wb(base + i * stride, ix, AXIS == 1 ? i : fixed, AXIS == 1 ? fixed : i, v[t].x, v[t].y, wb[t]);
        if (INVERSE) v[t].y = -v[t].y;
      }
#pragma unroll
      for (int t = 0; t < R1; ++t) ld.store_wb(base + (j1 + t * R2) * stride, ix, wb[t]);
    } else {
#pragma unroll
      for (int t = 0; t < R1; ++t) {
        const int i = j1 + t * R2;
        ld(base + i * stride, ix, AXIS == 1 ? i : fixed, AXIS == 1 ? fixed : i, v[t].x, v[t].y);
        if (INVERSE) v[t].y = -v[t].y;
      }
    }
    Dft<R1>::run(v);
#pragma unroll
    for (int t = 0; t < R1; ++t) buf[(j1 * R1 + t) * kFastL + l] = v[t];
  }
  group_sync(bar, TH);
  // stage 2: shared -> registers -> global
  for (int j2 = jj; j2 < R1; j2 += JS) {
    double2 v[R2];
#pragma unroll
    for (int t = 0; t < R2; ++t) v[t] = buf[(j2 + t * R1) * kFastL + l];
#pragma unroll
    for (int t = 1; t < R2; ++t) v[t] = cmul(v[t], G.tw[t * j2]);
    Dft<R2>::run(v);
    if constexpr (StoreOp::kSplitStore && R2 <= 8) {
      // an epilogue that reads further operands: every load and reduction first, then the stores (see above)
#pragma unroll
      for (int t = 0; t < R2; ++t) {
        const int i = j2 + t * R1;
        if (INVERSE) v[t].y = -v[t].y;
        st.accumulate(base + i * stride, ix, AXIS == 1 ? i : fixed, AXIS == 1 ? fixed : i, v[t]);
      }
#pragma unroll
      for (int t = 0; t < R2; ++t) st.put(base + (j2 + t * R1) * stride, v[t]);
    } else {
#pragma unroll
      for (int t = 0; t < R2; ++t) {
        const int i = j2 + t * R1;
        st.store(base + i * stride, ix, AXIS == 1 ? i : fixed, AXIS == 1 ? fixed : i, v[t].x, INVERSE ? -v[t].y : v[t].y);
      }
    }
  }
  group_sync(bar, TH);
}

template <int N, int AXIS, bool INVERSE, class LoadOp, class StoreOp>
__global__ void __launch_bounds__(fast_threads_yz<N>()) fft_yz_fast_kernel(FastGeom G, LoadOp ld_in, StoreOp st_in) {
  extern __shared__ double smem_raw[];
  LoadOp ld = ld_in;
  StoreOp st = st_in;
  pdl_launch_dependents();
  pdl_wait();
  if (G.stop && *G.stop) return;
  ld.begin(); st.begin();
  fft_yz_tile<N, AXIS, INVERSE, true>(G, ld, st, blockIdx.x, reinterpret_cast<double2 *>(smem_raw), threadIdx.x, 0);
  ld.finish(smem_raw);
  st.finish(smem_raw);
}

// ---- x passes: real lines <-> half spectrum ---------------------------------------------------------------
constexpr int kFastLP = 8;  // line pairs per block
// 256 threads: the FFT stages need only LP*max(R1,R2) <= 192 of them, the pointwise prologue/epilogue (Fermi-Dirac
// integrals, XC) uses all
template <int N> __host__ __device__ constexpr int fast_threads_x() { return 256; }
// plain x passes (no pointwise functor work): just the butterfly threads, and more resident blocks per SM instead
constexpr int kFastLPLight = 4;   // line pairs per block of the light configuration: half the tile, twice the blocks
template <int N> __host__ __device__ constexpr int fast_threads_x_light() {
  return kFastLPLight * (FastPlan<N>::R1 > FastPlan<N>::R2 ? FastPlan<N>::R1 : FastPlan<N>::R2);
}
template <int N> __host__ __device__ constexpr int fast_blocks_x_light() { return N >= 384 ? 6 : 8; }
template <int N> __host__ __device__ constexpr int fast_row_x() { return N + N / FastPlan<N>::R1; }   // padded smem row (elements)
template <int N> __device__ __forceinline__ int fast_pos(int i) { return i + i / FastPlan<N>::R1; }

// the two stages on the tile's LP complex lines held in shared memory (in place); t = thread index within the group
// of TH threads that owns the tile, bar = the group's barrier id (0 with the whole block)
template <int N, int TH, int LP = kFastLP>
__device__ __forceinline__ void fast_stages_x(double2 *buf, const double2 *tw, int t, int bar) {
  constexpr int R1 = FastPlan<N>::R1, R2 = FastPlan<N>::R2, ROW = fast_row_x<N>();
  static_assert(TH >= LP * R1 && TH >= LP * R2, "one butterfly per thread");
  {
    const int p = t / R2, j1 = t % R2;
    const bool act = t < LP * R2;
    double2 v[R1];
    if (act) {
#pragma unroll
      for (int q = 0; q < R1; ++q) v[q] = buf[p * ROW + fast_pos<N>(j1 + q * R2)];
      Dft<R1>::run(v);
    }
    group_sync(bar, TH);
    if (act) {
#pragma unroll
      for (int q = 0; q < R1; ++q) buf[p * ROW + j1 * (R1 + 1) + q] = v[q];   // = fast_pos(j1*R1 + q)
    }
  }
  group_sync(bar, TH);
  if (t < LP * R1) {
    const int p = t / R1, j2 = t % R1;
    double2 v[R2];
#pragma unroll
    for (int q = 0; q < R2; ++q) v[q] = buf[p * ROW + j2 + q * (R1 + 1)];       // = fast_pos(j2 + q*R1)
#pragma unroll
    for (int q = 1; q < R2; ++q) v[q] = cmul(v[q], tw[q * j2]);
    Dft<R2>::run(v);
#pragma unroll
    for (int q = 0; q < R2; ++q) buf[p * ROW + j2 + q * (R1 + 1)] = v[q];
  }
  group_sync(bar, TH);
}

// one x tile (8 pairs of real lines) by the whole block (256 threads); buf = [LP][ROW] shared
template <int N, bool PREFETCH, int TH = fast_threads_x<N>(), int LP = kFastLP, class LoadOp, class StoreOp>
__device__ __forceinline__ void fft_r2c_tile(const FastGeom &G, LoadOp &ld, StoreOp &st, int tile, double2 *buf,
                                             int tg = threadIdx.x, int bar = 0) {
  constexpr int ROW = fast_row_x<N>(), NXH = N / 2 + 1;
  const long long line0 = (long long)tile * (2 * LP);
  if (PREFETCH)
    for (int e = tg * 16; e < 2 * LP * N; e += TH * 16) ld.prefetch(line0 * N + e);   // contiguous real tile
  for (int e = tg; e < LP * N; e += TH) {
    const int p = e / N, i = e % N;
    const long long la = line0 + 2 * p, lb = la + 1;
    double a, b;
    ld.load_real2(la * N + i, lb * N + i, a, b);
    buf[p * ROW + fast_pos<N>(i)] = make_double2(a, b);
  }
  group_sync(bar, TH);
  fast_stages_x<N, TH, LP>(buf, G.tw, tg, bar);
  for (int e = tg; e < LP * G.P; e += TH) {
    const int p = e / G.P, k = e % G.P;
    const long long la = line0 + 2 * p, lb = la + 1;
    double2 A = make_double2(0.0, 0.0), B = A;
    if (k < NXH) {
      const double2 z = buf[p * ROW + fast_pos<N>(k)], m = buf[p * ROW + fast_pos<N>(k == 0 ? 0 : N - k)];
      A = make_double2(0.5 * (z.x + m.x), 0.5 * (z.y - m.y));
      B = make_double2(0.5 * (z.y + m.y), -0.5 * (z.x - m.x));
    }
    st.store(la * G.P + k, k, (int)(la % G.ny), (int)(la / G.ny), A.x, A.y);
    st.store(lb * G.P + k, k, (int)(lb % G.ny), (int)(lb / G.ny), B.x, B.y);
  }
  group_sync(bar, TH);
}

template <int N, bool PREFETCH, int TH = fast_threads_x<N>(), int LP = kFastLP, class LoadOp, class StoreOp>
__device__ __forceinline__ void fft_c2r_tile(const FastGeom &G, LoadOp &ld, StoreOp &st, int tile, double2 *buf,
                                             int tg = threadIdx.x, int bar = 0) {
  constexpr int ROW = fast_row_x<N>(), NXH = N / 2 + 1;
  const long long line0 = (long long)tile * (2 * LP);
  if (PREFETCH) {
    for (int e = tg * 8; e < 2 * LP * G.P; e += TH * 8) ld.prefetch(line0 * G.P + e);  // contiguous half tile
    for (int e = tg * 16; e < 2 * LP * N; e += TH * 16) st.prefetch(line0 * N + e);    // operands of the epilogue
  }
  for (int e = tg; e < LP * NXH; e += TH) {
    const int p = e / NXH, k = e % NXH;
    const long long la = line0 + 2 * p, lb = la + 1;
    double2 A, B;
    ld(la * G.P + k, k, (int)(la % G.ny), (int)(la / G.ny), A.x, A.y);
    ld(lb * G.P + k, k, (int)(lb % G.ny), (int)(lb / G.ny), B.x, B.y);
    buf[p * ROW + fast_pos<N>(k)] = make_double2(A.x - B.y, -(A.y + B.x));              // conj(A + i B)
    if (k > 0 && 2 * k < N) buf[p * ROW + fast_pos<N>(N - k)] = make_double2(A.x + B.y, A.y - B.x);  // conj(conj A + i conj B)
  }
  group_sync(bar, TH);
  fast_stages_x<N, TH, LP>(buf, G.tw, tg, bar);
  for (int e = tg; e < LP * N; e += TH) {
    const int p = e / N, i = e % N;
    const long long la = line0 + 2 * p, lb = la + 1;
    const double2 z = buf[p * ROW + fast_pos<N>(i)];
    st.store_real2(la * N + i, lb * N + i, z.x, -z.y);
  }
  group_sync(bar, TH);
}

template <int N, bool LIGHT, class LoadOp, class StoreOp>
__global__ void __launch_bounds__(LIGHT ? fast_threads_x_light<N>() : fast_threads_x<N>(), LIGHT ? fast_blocks_x_light<N>() : 1)
    fft_r2c_fast_kernel(FastGeom G, LoadOp ld_in, StoreOp st_in) {
  extern __shared__ double smem_raw[];
  LoadOp ld = ld_in;
  StoreOp st = st_in;
  pdl_launch_dependents();
  pdl_wait();
  if (G.stop && *G.stop) return;
  ld.begin(); st.begin();
  fft_r2c_tile<N, true, LIGHT ? fast_threads_x_light<N>() : fast_threads_x<N>(), LIGHT ? kFastLPLight : kFastLP>(
      G, ld, st, blockIdx.x, reinterpret_cast<double2 *>(smem_raw));
  ld.finish(smem_raw);
  st.finish(smem_raw);
}

template <int N, bool LIGHT, class LoadOp, class StoreOp>
__global__ void __launch_bounds__(LIGHT ? fast_threads_x_light<N>() : fast_threads_x<N>(), LIGHT ? fast_blocks_x_light<N>() : 1)
    fft_c2r_fast_kernel(FastGeom G, LoadOp ld_in, StoreOp st_in) {
  extern __shared__ double smem_raw[];
  LoadOp ld = ld_in;
  StoreOp st = st_in;
  pdl_launch_dependents();
  pdl_wait();
  if (G.stop && *G.stop) return;
  ld.begin(); st.begin();
  fft_c2r_tile<N, true, LIGHT ? fast_threads_x_light<N>() : fast_threads_x<N>(), LIGHT ? kFastLPLight : kFastLP>(
      G, ld, st, blockIdx.x, reinterpret_cast<double2 *>(smem_raw));
  ld.finish(smem_raw);
  st.finish(smem_raw);
}

// ---- register-centric x passes (plain passes of the streamed form) -----------------------------------------------
// The tile kernels above move every element through shared memory seven times (load, two in-place stages, Hermitian
// split: 112 bytes of shared-memory traffic per packed complex element against 16 bytes of HBM traffic) and were bound
// by the shared-memory data pipe (ncu, round 1: LSU data pipe 75%, x passes at 0.55-0.61 of the HBM peak while the y/z
// passes reach 0.75-0.9).  Here both stages live in registers like in the y/z kernels: stage 1 loads global memory
// straight into registers, one exchange through shared memory between the stages, stage 2 stores straight from
// registers -- and the Hermitian pairing z[k] <-> z[N-k] exchanges only the upper half of the spectrum (k >= N/2 is
// written, k <= N/2 reads its partner): 48 bytes of shared-memory traffic per element.
//   r2c: z = a + i b of two real lines;  A[k] = (z[k] + conj z[N-k])/2,  B[k] = (z[k] - conj z[N-k])/(2i),  k <= N/2.
//   c2r: z[k] = conj(A[k] + i B[k]), z[N-k] = conj(conj A[k] + i conj B[k]); forward stages; a = Re z, b = -Im z.
template <int N> __host__ __device__ constexpr int reg_threads_x() {
  return kFastLPLight * (FastPlan<N>::R1 > FastPlan<N>::R2 ? FastPlan<N>::R1 : FastPlan<N>::R2);
}
template <int N> __host__ __device__ constexpr int reg_blocks_x() { return N >= 384 ? 5 : (N >= 256 ? 6 : 8); }
// the r2c kernel needs all 2 R1 stage-1 loads of a thread in flight at once (168 registers at N = 384: with 126 ptxas
// consumed the first loads before it issued the last and the HBM latency was paid three to four times per tile)
template <int N> __host__ __device__ constexpr int reg_blocks_r2c() { return N >= 384 ? 4 : (N >= 192 ? 5 : 8); }

template <int N, class LoadOp, class StoreOp>
__global__ void __launch_bounds__(reg_threads_x<N>(), reg_blocks_r2c<N>()) fft_r2c_reg_kernel(FastGeom G, LoadOp ld_in, StoreOp st_in) {
  constexpr int R1 = FastPlan<N>::R1, R2 = FastPlan<N>::R2, ROW = fast_row_x<N>(), LP = kFastLPLight;
  static_assert(R2 % 2 == 0, "the Hermitian exchange splits stage-2 outputs at q = R2/2");
  extern __shared__ double smem_raw[];
  double2 *buf = reinterpret_cast<double2 *>(smem_raw);   // [LP][ROW]
  LoadOp ld = ld_in;
  StoreOp st = st_in;
  pdl_launch_dependents();
  pdl_wait();
  if (G.stop && *G.stop) return;
  ld.begin(); st.begin();
  const int t = threadIdx.x;
  const long long line0 = (long long)blockIdx.x * (2 * LP);
  if (t < LP * R2) {   // stage 1: global -> registers -> shared
    const int p = t / R2, j1 = t % R2;
    const long long la = (line0 + 2 * p) * N, lb = la + N;
    double2 v[R1];
#pragma unroll
    for (int q = 0; q < R1; ++q) ld.load_real2(la + j1 + q * R2, lb + j1 + q * R2, v[q].x, v[q].y);
    Dft<R1>::run(v);
#pragma unroll
    for (int q = 0; q < R1; ++q) buf[p * ROW + j1 * (R1 + 1) + q] = v[q];
  }
  __syncthreads();
  const bool act = t < LP * R1;
  const int p = t / R1, j2 = t % R1;
  double2 v[R2];
  if (act) {           // stage 2: shared -> registers; v[q] = z[j2 + q R1]
#pragma unroll
    for (int q = 0; q < R2; ++q) v[q] = buf[p * ROW + j2 + q * (R1 + 1)];
#pragma unroll
    for (int q = 1; q < R2; ++q) v[q] = cmul(v[q], G.tw[q * j2]);
    Dft<R2>::run(v);
  }
  __syncthreads();
  if (act) {           // upper half of the spectrum (k >= N/2) to shared memory, natural order
#pragma unroll
    for (int q = R2 / 2; q < R2; ++q) buf[p * ROW + j2 + q * R1] = v[q];
  }
  __syncthreads();
  if (act) {           // k <= N/2 takes its partner z[N-k] and stores A[k], B[k] straight from registers
    const long long la = line0 + 2 * p, lb = la + 1;
    const int iya = (int)(la % G.ny), iza = (int)(la / G.ny), iyb = (int)(lb % G.ny), izb = (int)(lb / G.ny);
#pragma unroll
    for (int q = 0; q <= R2 / 2; ++q) {
      if (q == R2 / 2 && j2 != 0) break;          // k = N/2 belongs to j2 = 0 only
      const int k = j2 + q * R1;
      const double2 z = v[q], m = k == 0 ? v[0] : buf[p * ROW + (N - k)];
      st.store(la * G.P + k, k, iya, iza, 0.5 * (z.x + m.x), 0.5 * (z.y - m.y));
      st.store(lb * G.P + k, k, iyb, izb, 0.5 * (z.y + m.y), -0.5 * (z.x - m.x));
    }
  }
  ld.finish(smem_raw);
  st.finish(smem_raw);
}

// The same pass with its input brought in by the copy engine (plain real input only).  ncu of fft_r2c_reg_kernel<384>:
// long_scoreboard 8.3 warps per issue, 17% warps, 0.67 of the HBM peak -- 3072 eight-byte loads per block have to be issued
// by 96 threads before the first butterfly can start.  The 2 LP real lines of a block are ONE contiguous run
// (2 LP N doubles): a single cp.async.bulk completing on an mbarrier brings it into shared memory, stage 1 reads its
// operands from there (LDS.64, conflict-free), the rest is the kernel above.
template <int N, class StoreOp>
__global__ void __launch_bounds__(reg_threads_x<N>(), reg_blocks_r2c<N>()) fft_r2c_tma_kernel(FastGeom G, const double *__restrict__ src, StoreOp st_in) {
  constexpr int R1 = FastPlan<N>::R1, R2 = FastPlan<N>::R2, ROW = fast_row_x<N>(), LP = kFastLPLight;
  static_assert(R2 % 2 == 0, "the Hermitian exchange splits stage-2 outputs at q = R2/2");
  extern __shared__ double smem_raw[];
  double2 *buf = reinterpret_cast<double2 *>(smem_raw);   // [LP][ROW]
  double *s_in = smem_raw + 2 * LP * ROW;                  // [2 LP][N]
  __shared__ unsigned long long s_bar;
  StoreOp st = st_in;
  pdl_launch_dependents();
  const int t = threadIdx.x;
  const long long line0 = (long long)blockIdx.x * (2 * LP);
  if (t == 0) mbar_init(&s_bar, 1);
  pdl_wait();
  if (G.stop && *G.stop) return;
  if (t == 0) {
    mbar_arrive_expect_tx(&s_bar, (unsigned)(2 * LP * N * sizeof(double)));
    bulk_copy_g2s(s_in, src + line0 * N, (unsigned)(2 * LP * N * sizeof(double)), &s_bar);
  }
  st.begin();
  __syncthreads();   // the barrier is initialised
  mbar_wait(&s_bar, 0);
  if (t < LP * R2) {   // stage 1: shared -> registers -> shared
    const int p = t / R2, j1 = t % R2;
    const double *la = s_in + (2 * p) * N, *lb = la + N;
    double2 v[R1];
#pragma unroll
    for (int q = 0; q < R1; ++q) v[q] = make_double2(la[j1 + q * R2], lb[j1 + q * R2]);
    Dft<R1>::run(v);
#pragma unroll
    for (int q = 0; q < R1; ++q) buf[p * ROW + j1 * (R1 + 1) + q] = v[q];
  }
  __syncthreads();
  const bool act = t < LP * R1;
  const int p = t / R1, j2 = t % R1;
  double2 v[R2];
  if (act) {           // stage 2: shared -> registers; v[q] = z[j2 + q R1]
#pragma unroll
    for (int q = 0; q < R2; ++q) v[q] = buf[p * ROW + j2 + q * (R1 + 1)];
#pragma unroll
    for (int q = 1; q < R2; ++q) v[q] = cmul(v[q], G.tw[q * j2]);
    Dft<R2>::run(v);
  }
  __syncthreads();
  if (act) {           // upper half of the spectrum (k >= N/2) to shared memory, natural order
#pragma unroll
    for (int q = R2 / 2; q < R2; ++q) buf[p * ROW + j2 + q * R1] = v[q];
  }
  __syncthreads();
  if (act) {           // k <= N/2 takes its partner z[N-k] and stores A[k], B[k] straight from registers
    const long long la = line0 + 2 * p, lb = la + 1;
    const int iya = (int)(la % G.ny), iza = (int)(la / G.ny), iyb = (int)(lb % G.ny), izb = (int)(lb / G.ny);
#pragma unroll
    for (int q = 0; q <= R2 / 2; ++q) {
      if (q == R2 / 2 && j2 != 0) break;          // k = N/2 belongs to j2 = 0 only
      const int k = j2 + q * R1;
      const double2 z = v[q], m = k == 0 ? v[0] : buf[p * ROW + (N - k)];
      st.store(la * G.P + k, k, iya, iza, 0.5 * (z.x + m.x), 0.5 * (z.y - m.y));
      st.store(lb * G.P + k, k, iyb, izb, 0.5 * (z.y + m.y), -0.5 * (z.x - m.x));
    }
  }
  st.finish(smem_raw);
}

template <int N, class LoadOp, class StoreOp>
__global__ void __launch_bounds__(reg_threads_x<N>(), reg_blocks_x<N>()) fft_c2r_reg_kernel(FastGeom G, LoadOp ld_in, StoreOp st_in) {
  constexpr int R1 = FastPlan<N>::R1, R2 = FastPlan<N>::R2, ROW = fast_row_x<N>(), LP = kFastLPLight;
  static_assert(R1 % 2 == 0, "the Hermitian exchange splits stage-1 inputs at q = R1/2");
  extern __shared__ double smem_raw[];
  double2 *buf = reinterpret_cast<double2 *>(smem_raw);   // [LP][ROW]
  LoadOp ld = ld_in;
  StoreOp st = st_in;
  pdl_launch_dependents();
  pdl_wait();
  if (G.stop && *G.stop) return;
  ld.begin(); st.begin();
  const int t = threadIdx.x;
  const long long line0 = (long long)blockIdx.x * (2 * LP);
  const bool act1 = t < LP * R2;
  const int p1 = t / R2, j1 = t % R2;
  double2 v1[R1];
  if (act1) {          // i = j1 + q R2 <= N/2: load A[i], B[i]; keep z[i], hand z[N-i] to its owner through shared memory
    const long long la = line0 + 2 * p1, lb = la + 1;
    const int iya = (int)(la % G.ny), iza = (int)(la / G.ny), iyb = (int)(lb % G.ny), izb = (int)(lb / G.ny);
#pragma unroll
    for (int q = 0; q <= R1 / 2; ++q) {
      if (q == R1 / 2 && j1 != 0) break;          // i = N/2 belongs to j1 = 0 only
      const int i = j1 + q * R2;
      double2 A, B;
      ld(la * G.P + i, i, iya, iza, A.x, A.y);
      ld(lb * G.P + i, i, iyb, izb, B.x, B.y);
      v1[q] = make_double2(A.x - B.y, -(A.y + B.x));                                         // conj(A + i B)
      if (i > 0 && 2 * i < N) buf[p1 * ROW + (N - i)] = make_double2(A.x + B.y, A.y - B.x);   // conj(conj A + i conj B)
    }
  }
  __syncthreads();
  if (act1) {
#pragma unroll
    for (int q = R1 / 2; q < R1; ++q) {
      if (q == R1 / 2 && j1 == 0) continue;       // loaded above
      v1[q] = buf[p1 * ROW + j1 + q * R2];
    }
    Dft<R1>::run(v1);
  }
  __syncthreads();
  if (act1) {
#pragma unroll
    for (int q = 0; q < R1; ++q) buf[p1 * ROW + j1 * (R1 + 1) + q] = v1[q];
  }
  __syncthreads();
  if (t < LP * R1) {   // stage 2: shared -> registers -> global (real lines)
    const int p = t / R1, j2 = t % R1;
    const long long la = (line0 + 2 * p) * N, lb = la + N;
    double2 v[R2];
#pragma unroll
    for (int q = 0; q < R2; ++q) v[q] = buf[p * ROW + j2 + q * (R1 + 1)];
#pragma unroll
    for (int q = 1; q < R2; ++q) v[q] = cmul(v[q], G.tw[q * j2]);
    Dft<R2>::run(v);
#pragma unroll
    for (int q = 0; q < R2; ++q) st.store_real2(la + j2 + q * R1, lb + j2 + q * R1, v[q].x, -v[q].y);
  }
  ld.finish(smem_raw);
  st.finish(smem_raw);
}

// ---- host dispatch ------------------------------------------------------------------------------------------
template <int N, int AXIS, bool INVERSE, class LoadOp, class StoreOp>
static inline cudaError_t fft_launch_yz_fast_n(const FastGeom &G, LoadOp ld, StoreOp st, cudaStream_t stream) {
  auto kern = fft_yz_fast_kernel<N, AXIS, INVERSE, LoadOp, StoreOp>;
  size_t smem = sizeof(double2) * N * kFastL;
  if (smem < 4096) smem = 4096;
  static int attr_dev = -1;   // the opt-in is per device: set it again when the calling thread's device differs
  int dev = 0;
  cudaGetDevice(&dev);
  if (attr_dev != dev) {
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, 64 * 1024);
    if (e != cudaSuccess) return e;
    attr_dev = dev;
  }
  const unsigned blocks = (unsigned)((AXIS == 1 ? G.nz : G.ny) * (G.P / kFastL));
  void *args[] = {(void *)&G, (void *)&ld, (void *)&st};
  return launch_maybe_pdl((const void *)kern, dim3(blocks), dim3(fast_threads_yz<N>()), args, smem, stream, G.pdl != 0);
}
// returns cudaErrorNotSupported when the axis length has no fast plan (caller falls back to the generic pass)
template <int AXIS, bool INVERSE, class LoadOp, class StoreOp>
static inline cudaError_t fft_launch_yz_fast(int n, const FastGeom &G, LoadOp ld, StoreOp st, cudaStream_t stream) {
  switch (n) {
    case 32: return fft_launch_yz_fast_n<32, AXIS, INVERSE>(G, ld, st, stream);
    case 64: return fft_launch_yz_fast_n<64, AXIS, INVERSE>(G, ld, st, stream);
    case 128: return fft_launch_yz_fast_n<128, AXIS, INVERSE>(G, ld, st, stream);
    case 192: return fft_launch_yz_fast_n<192, AXIS, INVERSE>(G, ld, st, stream);
    case 256: return fft_launch_yz_fast_n<256, AXIS, INVERSE>(G, ld, st, stream);
    case 384: return fft_launch_yz_fast_n<384, AXIS, INVERSE>(G, ld, st, stream);
    default: return cudaErrorNotSupported;
  }
}

template <int N, bool INVERSE, bool LIGHT, class LoadOp, class StoreOp>
static inline cudaError_t fft_launch_x_fast_n(const FastGeom &G, LoadOp ld, StoreOp st, cudaStream_t stream) {
  constexpr int LP = LIGHT ? kFastLPLight : kFastLP;
  size_t smem = sizeof(double2) * LP * fast_row_x<N>();
  if (smem < 4096) smem = 4096;
  const unsigned blocks = (unsigned)((long long)G.ny * G.nz / (2 * LP));
  constexpr int TH = LIGHT ? reg_threads_x<N>() : fast_threads_x<N>();
  static int attr_dev = -1;
  int dev = 0;
  cudaGetDevice(&dev);
  const bool attr_set = attr_dev == dev;
  const void *kern;
  if constexpr (!INVERSE && LIGHT && std::is_same<LoadOp, LoadReal>::value) {
    if (G.tma) {   // input through the copy engine
      auto tk = fft_r2c_tma_kernel<N, StoreOp>;
      const size_t tsmem = sizeof(double2) * LP * fast_row_x<N>() + sizeof(double) * 2 * LP * N;
      static int tattr_dev = -1;
      if (tattr_dev != dev) {
        cudaError_t e = cudaFuncSetAttribute(tk, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)tsmem);
        if (e != cudaSuccess) return e;
        tattr_dev = dev;
      }
      const double *srcp = ld.src;
      void *targs[] = {(void *)&G, (void *)&srcp, (void *)&st};
      return launch_maybe_pdl((const void *)tk, dim3(blocks), dim3(TH), targs, tsmem, stream, G.pdl != 0);
    }
  }
  if constexpr (INVERSE) {
    if constexpr (LIGHT) kern = (const void *)fft_c2r_reg_kernel<N, LoadOp, StoreOp>;
    else kern = (const void *)fft_c2r_fast_kernel<N, false, LoadOp, StoreOp>;
  } else {
    if constexpr (LIGHT) kern = (const void *)fft_r2c_reg_kernel<N, LoadOp, StoreOp>;
    else kern = (const void *)fft_r2c_fast_kernel<N, false, LoadOp, StoreOp>;
  }
  if (!attr_set) {
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, 64 * 1024);
    if (e != cudaSuccess) return e;
    attr_dev = dev;
  }
  void *args[] = {(void *)&G, (void *)&ld, (void *)&st};
  return launch_maybe_pdl(kern, dim3(blocks), dim3(TH), args, smem, stream, G.pdl != 0);
}
// LIGHT: the functors do no arithmetic worth extra threads (plain loads/stores): butterfly threads only, 3-4 blocks per SM
template <bool INVERSE, bool LIGHT, class LoadOp, class StoreOp>
static inline cudaError_t fft_launch_x_fast(int n, const FastGeom &G, LoadOp ld, StoreOp st, cudaStream_t stream) {
  if (((long long)G.ny * G.nz) % (2 * kFastLP) != 0) return cudaErrorNotSupported;
  switch (n) {
    case 32: return fft_launch_x_fast_n<32, INVERSE, LIGHT>(G, ld, st, stream);
    case 64: return fft_launch_x_fast_n<64, INVERSE, LIGHT>(G, ld, st, stream);
    case 128: return fft_launch_x_fast_n<128, INVERSE, LIGHT>(G, ld, st, stream);
    case 192: return fft_launch_x_fast_n<192, INVERSE, LIGHT>(G, ld, st, stream);
    case 256: return fft_launch_x_fast_n<256, INVERSE, LIGHT>(G, ld, st, stream);
    case 384: return fft_launch_x_fast_n<384, INVERSE, LIGHT>(G, ld, st, stream);
    default: return cudaErrorNotSupported;
  }
}

}  // namespace arche
