// common.cuh -- shared device helpers of the B200 path (sm_100a, fp64).
// Deterministic reductions: warp shuffles -> block partials -> the last-arriving block sums all block
// partials in index order (fixed order => bit-reproducible; no fp64 atomics in any value path).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#define ARCHE_PI 3.14159265358979323846264338327950288

namespace arche {

constexpr int kMaxRed = 8;        // max simultaneous sums per reduction

struct GridGeom {
  int nx, ny, nz;
  int nxh, P;                     // half spectrum: nxh = nx/2+1 stored columns, row pitch P (multiple of 8)
  long long ng, nh;               // real points nx*ny*nz; half-spectrum elements P*ny*nz
  double Lx, Ly, Lz, vol, dV;
  const double *kx, *ky, *kz;     // k components per storage index, device
  const double *kx2, *ky2, *kz2;  // squares
};

// L2 prefetch of the 128-byte line holding *p: the fused passes request every operand line of a tile up front, so
// the later (register-limited, partly serialised) loads find their data in L2 instead of paying HBM latency each
__device__ __forceinline__ void prefetch_l2(const void *p) { asm volatile("prefetch.global.L2 [%0];" ::"l"(p)); }

// ---- sm_90+/sm_100a launch and copy primitives (inline PTX) --------------------------------------------------------
// Programmatic dependent launch: a kernel launched with cudaLaunchAttributeProgrammaticStreamSerialization may start
// while its predecessor in the stream is still draining.  Every such kernel calls pdl_launch_dependents() first (its own
// successor may be scheduled as soon as all of its blocks are resident), does the work that does not depend on the
// predecessor (index arithmetic, the Fermi-Dirac table copy), and calls pdl_wait() before it touches anything an earlier
// kernel wrote -- the wait returns when the predecessor grid has completed and its writes are visible.  Both are
// no-ops in a kernel launched without the attribute.
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

// Bulk asynchronous copy global -> shared (the 1D form of the tensor memory accelerator, cp.async.bulk) completing on
// an mbarrier: one thread issues the copy, the copy engine moves the bytes without passing through registers or the
// LSU, every thread waits on the barrier's phase.  Sizes and addresses are multiples of 16 bytes.
__device__ __forceinline__ unsigned smem_addr_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long *bar, unsigned arrivals) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_addr_u32(bar)), "r"(arrivals) : "memory");
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // make the initialised barrier visible to the copy engine
}
// orders this thread's earlier generic-proxy writes to shared memory before later writes of the copy engine (async
// proxy) to the same addresses: call it after clearing a buffer that bulk copies will fill, before the block barrier
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void mbar_arrive_expect_tx(unsigned long long *bar, unsigned bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_addr_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_copy_g2s(void *smem_dst, const void *gmem_src, unsigned bytes, unsigned long long *bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_addr_u32(smem_dst)),
               "l"(gmem_src), "r"(bytes), "r"(smem_addr_u32(bar))
               : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long *bar, unsigned parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "MBAR_WAIT:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra MBAR_DONE;\n"
      "bra MBAR_WAIT;\n"
      "MBAR_DONE:\n"
      "}\n" ::"r"(smem_addr_u32(bar)),
      "r"(parity)
      : "memory");
}

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}
__device__ __forceinline__ double warp_min(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = fmin(v, __shfl_xor_sync(0xffffffffu, v, o));
  return v;
}
__device__ __forceinline__ double warp_max(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
  return v;
}

// op: 0 sum, 1 min, 2 max
__device__ __forceinline__ double red_combine(double a, double b, int op) {
  return op == 0 ? a + b : (op == 1 ? fmin(a, b) : fmax(a, b));
}
__device__ __forceinline__ double warp_red(double v, int op) {
  return op == 0 ? warp_sum(v) : (op == 1 ? warp_min(v) : warp_max(v));
}

// Block-level reduction of NQ quantities; result valid in thread 0.  Block size <= 1024.
template <int NQ>
__device__ __forceinline__ void block_reduce(double (&v)[NQ], const int (&op)[NQ], double *smem /*[NQ*32]*/) {
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
#pragma unroll
  for (int q = 0; q < NQ; ++q) {
    double x = warp_red(v[q], op[q]);
    if (lane == 0) smem[q * 32 + wid] = x;
  }
  __syncthreads();
  if (wid == 0) {
#pragma unroll
    for (int q = 0; q < NQ; ++q) {
      double ident = op[q] == 0 ? 0.0 : (op[q] == 1 ? 1.0e308 : -1.0e308);
      double x = lane < nw ? smem[q * 32 + lane] : ident;
      v[q] = warp_red(x, op[q]);
    }
  }
  __syncthreads();
}

// Barrier-based form of the grid reduction for cooperative kernels: every block writes its partials, the caller
// issues a grid barrier, then every block sums all partials in the same fixed order (no atomics, no last-block
// serialisation; all blocks end up with identical totals).  Partials are stored [quantity][block] so that a warp
// reads one quantity of 32 blocks as one contiguous 256-byte segment.
template <int NQ>
__device__ __forceinline__ void block_partials(double (&v)[NQ], const int (&op)[NQ], double *smem /*[NQ*32]*/,
                                               double *out /*[stride][gridDim.x]*/, int stride = NQ, int offset = 0) {
  (void)stride;
  block_reduce<NQ>(v, op, smem);
  if (threadIdx.x == 0) {
#pragma unroll
    for (int q = 0; q < NQ; ++q) out[(size_t)(offset + q) * gridDim.x + blockIdx.x] = v[q];
  }
}
// totals valid in every thread (t[NQ]); call after the grid barrier that follows block_partials.  Warp q sums
// quantity q over the blocks: the loads of up to 160 blocks are issued together (one L2 round trip), then one
// shuffle tree; needs NQ <= 2 x warps per block.
template <int NQ>
__device__ __forceinline__ void block_totals(const int (&op)[NQ], const double *in /*[NQ][gridDim.x]*/, double *smem,
                                             double (&t)[NQ]) {
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = blockDim.x >> 5;
  const unsigned int G = gridDim.x;
  for (int q = wid; q < NQ; q += nw) {
    const int o = op[q];
    const double ident = o == 0 ? 0.0 : (o == 1 ? 1.0e308 : -1.0e308);
    const double *row = in + (size_t)q * G;
    double v[5];
#pragma unroll
    for (int k = 0; k < 5; ++k) { const unsigned int b = lane + 32 * k; v[k] = b < G ? __ldcg(row + b) : ident; }
    double a = v[0];
#pragma unroll
    for (int k = 1; k < 5; ++k) a = red_combine(a, v[k], o);
    for (unsigned int b = lane + 160; b < G; b += 32) a = red_combine(a, __ldcg(row + b), o);
    a = warp_red(a, o);
    if (lane == 0) smem[q] = a;
  }
  __syncthreads();
#pragma unroll
  for (int q = 0; q < NQ; ++q) t[q] = smem[q];
  __syncthreads();
}

// Grid-level deterministic reduction.  Every block calls this once with its per-thread values.
// partials: [gridDim.x * NQ]; counter: zero before the launch (reset by the last block);
// returns true in ALL threads of the last block, with the totals in `out` (shared memory, [NQ]).
template <int NQ>
__device__ __forceinline__ bool grid_reduce(double (&v)[NQ], const int (&op)[NQ], double *partials,
                                            unsigned int *counter, double *smem /*[NQ*32 + NQ]*/) {
  block_reduce<NQ>(v, op, smem);
  __shared__ bool s_last;
  if (threadIdx.x == 0) {
#pragma unroll
    for (int q = 0; q < NQ; ++q) partials[(size_t)blockIdx.x * NQ + q] = v[q];
    __threadfence();
    unsigned int t = atomicAdd(counter, 1u);
    s_last = (t == gridDim.x - 1);
  }
  __syncthreads();
  if (!s_last) return false;
  __threadfence();
  // fixed-order sum over blocks: thread t takes blocks t, t+B, ... (order independent of which block is last)
  double acc[NQ];
#pragma unroll
  for (int q = 0; q < NQ; ++q) acc[q] = op[q] == 0 ? 0.0 : (op[q] == 1 ? 1.0e308 : -1.0e308);
  for (unsigned int b = threadIdx.x; b < gridDim.x; b += blockDim.x) {
#pragma unroll
    for (int q = 0; q < NQ; ++q) acc[q] = red_combine(acc[q], __ldcg(&partials[(size_t)b * NQ + q]), op[q]);
  }
  block_reduce<NQ>(acc, op, smem);
  if (threadIdx.x == 0) {
#pragma unroll
    for (int q = 0; q < NQ; ++q) smem[NQ * 32 + q] = acc[q];
    *counter = 0u;
  }
  __syncthreads();
  return true;
}

}  // namespace arche
