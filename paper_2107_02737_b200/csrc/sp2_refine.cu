// sp2_refine.cu -- optional FP64 refinement layers.
//
// "We may also add two extra layers in Eq. (19), with a higher-order double-precision (64 bit)
// representation of X in the activation function, which then acts as a refinement step, where the eigenvalues
// are purified to be closer to exactly 1 and 0" (effect on the forces: Fig. 3-4).
//
// After the FP16 hi/lo layer stack has stopped, the final iterate X_L = c I + (Yh + Ym) 2^-t is expanded to
// float64 and `refine_layers` more SP2 layers X <- X^2 or 2X - X^2 (same trace rule) run in float64 on the
// FP64 tensor path (mma.sync m8n8k4 f64: tcgen05 has no FP64 kind).  X is symmetric, so only tiles on or above
// the diagonal are computed and mirrored, and B[k][j] = X[j][k] makes both operands row panels of X.
//
//   k_refine_expand    planes -> X (float64, npad x npad, zero padding), partial tr X and ||X||_F^2
//   k_refine_layer     one layer: 128x128 tiles, 3-stage cp.async ring, DMMA, fused update + mirrored store +
//                      partials; the last block reduces them and fixes the next branch
//   k_refine_finalise  X -> D in the caller's dtype, tr(DH); result struct
#include <cuda_runtime.h>
#include <cuda_fp16.h>
#include <stdint.h>
#include "sp2_internal.cuh"

namespace {

constexpr int kT = 128;          // tile edge
constexpr int kK = 16;           // k doubles per stage
constexpr int kLd = 20;          // padded row pitch of a stage tile in doubles (160 B: 16-B aligned, conflict-free LDS.64)
constexpr int kRStages = 3;
constexpr int kTileDoubles = kT * kLd;

__device__ __forceinline__ void cp_async16(void* smem, const void* gmem) {
  const uint32_t s = (uint32_t)__cvta_generic_to_shared(smem);
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(s), "l"(gmem) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

__device__ __forceinline__ void dmma(double& d0, double& d1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0, %1}, {%2}, {%3}, {%0, %1};"
               : "+d"(d0), "+d"(d1)
               : "d"(a), "d"(b));
}

__device__ __forceinline__ double block_sum(double v, double* sh /* 8 */) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  __syncthreads();
  if (lane == 0) sh[warp] = v;
  __syncthreads();
  double t = 0.0;
  for (int w = 0; w < (int)(blockDim.x >> 5); ++w) t += sh[w];
  return t;
}

// tr X and ||X||_F^2 decide the branch exactly like the FP16 controller (reading R3)
__device__ inline void refine_decide(Sp2Ctrl* c, double tr_x, double fro_x) {
  const double nocc = (double)c->n_occ;
  c->ref_tr = tr_x;
  c->ref_fro = fro_x;
  c->ref_plus = fabs(fro_x - nocc) < fabs(2.0 * tr_x - fro_x - nocc) ? 1 : 0;
}

__device__ inline bool refine_active(const Sp2Ctrl* c) {
  return c->done && (c->status == SP2_OK || c->status == SP2_WARN_NOT_CONVERGED);
}

// ------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_refine_expand(Sp2Ctrl* c, const __half* Yh0, const __half* Ym0,
                                                       const __half* Yh1, const __half* Ym1, int npad,
                                                       double* __restrict__ X, double* __restrict__ slots) {
  if (!refine_active(c)) return;
  const int par = c->n & 1;
  const __half* Yh = par ? Yh1 : Yh0;
  const __half* Ym = par ? Ym1 : Ym0;
  const double sy = sp2_exp2i(-c->t), shift = c->c;
  const int N = c->N;
  const int row = blockIdx.x;
  double tr = 0.0, fro = 0.0;
  for (int j = threadIdx.x; j < npad; j += 256) {
    double x = 0.0;
    if (row < N && j < N) {
      x = (double)(__half2float(Yh[(size_t)row * npad + j]) + __half2float(Ym[(size_t)row * npad + j])) * sy;
      if (j == row) { x += shift; tr += x; }
      fro += x * x;
    }
    X[(size_t)row * npad + j] = x;
  }
  __shared__ double sh[8];
  tr = block_sum(tr, sh);
  fro = block_sum(fro, sh);
  if (threadIdx.x == 0) { slots[2 * row] = tr; slots[2 * row + 1] = fro; }
}

// reduce `count` (tr, fro) slot pairs in index order, one block
__global__ void __launch_bounds__(256) k_refine_reduce(Sp2Ctrl* c, const double* slots, int count) {
  if (!refine_active(c)) return;
  __shared__ double sh[8];
  double a = 0.0, b = 0.0;
  for (int i = threadIdx.x; i < count; i += 256) { a += slots[2 * i]; b += slots[2 * i + 1]; }
  a = block_sum(a, sh);
  b = block_sum(b, sh);
  if (threadIdx.x == 0) refine_decide(c, a, b);
}

// ------------------------------------------------------------------------------------------
// One float64 layer.  Block = one upper-triangular 128x128 tile; 8 warps as 2 (rows) x 4 (cols), warp tile 64x32 =
// 8 x 4 DMMA tiles of 8x8 (64 accumulator doubles per thread).
__global__ void __launch_bounds__(256, 1) k_refine_layer(Sp2Ctrl* c, const double* __restrict__ Xin, double* __restrict__ Xout,
                                                         int npad, double* __restrict__ slots, unsigned int* ticket) {
  if (!refine_active(c)) return;
  extern __shared__ double rsm[];
  const int nb = npad / kT;
  int bi = 0, rem = blockIdx.x;
  while (rem >= nb - bi) { rem -= nb - bi; ++bi; }
  const int bj = bi + rem;
  const int i0 = bi * kT, j0 = bj * kT;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int wm = warp >> 2, wn = warp & 3;                 // 2 x 4 warps
  const int g = lane >> 2, q = lane & 3;                   // DMMA fragment coordinates

  auto stage_a = [&](int s) { return rsm + (size_t)s * 2 * kTileDoubles; };
  auto stage_b = [&](int s) { return rsm + (size_t)s * 2 * kTileDoubles + kTileDoubles; };
  auto load_stage = [&](int s, int kb) {
    // 128 rows x 16 doubles per operand = 1024 chunks of 16 B; 4 + 4 per thread
#pragma unroll
    for (int t = 0; t < 4; ++t) {
      const int ch = tid + t * 256;
      const int r = ch >> 3, cc = (ch & 7) * 2;
      cp_async16(stage_a(s) + r * kLd + cc, Xin + (size_t)(i0 + r) * npad + kb * kK + cc);
      cp_async16(stage_b(s) + r * kLd + cc, Xin + (size_t)(j0 + r) * npad + kb * kK + cc);
    }
    cp_async_commit();
  };

  double acc[8][4][2];
#pragma unroll
  for (int a = 0; a < 8; ++a)
#pragma unroll
    for (int b = 0; b < 4; ++b) { acc[a][b][0] = 0.0; acc[a][b][1] = 0.0; }

  const int KB = npad / kK;
  load_stage(0, 0);
  if (KB > 1) load_stage(1, 1); else cp_async_commit();
  for (int kb = 0; kb < KB; ++kb) {
    cp_async_wait<1>();
    __syncthreads();
    if (kb + 2 < KB) load_stage((kb + 2) % kRStages, kb + 2); else cp_async_commit();
    const double* A = stage_a(kb % kRStages) + (wm * 64) * kLd;
    const double* B = stage_b(kb % kRStages) + (wn * 32) * kLd;
#pragma unroll
    for (int k4 = 0; k4 < kK / 4; ++k4) {
      double af[8], bf[4];
#pragma unroll
      for (int a = 0; a < 8; ++a) af[a] = A[(a * 8 + g) * kLd + k4 * 4 + q];
#pragma unroll
      for (int b = 0; b < 4; ++b) bf[b] = B[(b * 8 + g) * kLd + k4 * 4 + q];
#pragma unroll
      for (int a = 0; a < 8; ++a)
#pragma unroll
        for (int b = 0; b < 4; ++b) dmma(acc[a][b][0], acc[a][b][1], af[a], bf[b]);
    }
  }
  cp_async_wait<0>();

  // epilogue: X' = X^2 or 2X - X^2; elements with gj >= gi only, mirrored; partials
  const bool plus = c->ref_plus != 0;
  double tr = 0.0, fro = 0.0;
#pragma unroll
  for (int a = 0; a < 8; ++a) {
    const int gi = i0 + wm * 64 + a * 8 + g;
#pragma unroll
    for (int b = 0; b < 4; ++b) {
#pragma unroll
      for (int e = 0; e < 2; ++e) {
        const int gj = j0 + wn * 32 + b * 8 + 2 * q + e;
        if (gj < gi) continue;
        double v = acc[a][b][e];
        if (!plus) v = 2.0 * Xin[(size_t)gi * npad + gj] - v;
        Xout[(size_t)gi * npad + gj] = v;
        if (gj > gi) { Xout[(size_t)gj * npad + gi] = v; fro += 2.0 * v * v; }
        else { tr += v; fro += v * v; }
      }
    }
  }
  __shared__ double sh[8];
  __shared__ unsigned int is_last;
  tr = block_sum(tr, sh);
  fro = block_sum(fro, sh);
  if (tid == 0) {
    slots[2 * blockIdx.x] = tr; slots[2 * blockIdx.x + 1] = fro;
    __threadfence();
    is_last = (atomicAdd(ticket, 1u) == gridDim.x - 1) ? 1u : 0u;
  }
  __syncthreads();
  if (!is_last) return;
  __threadfence();
  double a = 0.0, b = 0.0;
  for (int i = tid; i < (int)gridDim.x; i += 256) { a += __ldcg(slots + 2 * i); b += __ldcg(slots + 2 * i + 1); }
  a = block_sum(a, sh);
  b = block_sum(b, sh);
  if (tid == 0) { *ticket = 0u; refine_decide(c, a, b); c->ref_done += 1; }
}

// ------------------------------------------------------------------------------------------
template <typename TI, typename TO>
__global__ void __launch_bounds__(256) k_refine_finalise(const Sp2Ctrl* __restrict__ c, const double* __restrict__ X, int npad,
                                                         const TI* __restrict__ H, long ldh, TO* __restrict__ D, long ldo,
                                                         double* __restrict__ slots) {
  if (!refine_active(c)) return;
  const int N = c->N, row = blockIdx.x;
  double trdh = 0.0;
  for (int j = threadIdx.x; j < N; j += 256) {
    const double x = X[(size_t)row * npad + j];
    D[(size_t)row * ldo + j] = (TO)x;
    trdh += x * (double)H[(size_t)row * ldh + j];
  }
  __shared__ double sh[8];
  trdh = block_sum(trdh, sh);
  if (threadIdx.x == 0) slots[row] = trdh;
}

__global__ void __launch_bounds__(256) k_refine_result(Sp2Ctrl* c, const double* slots, int count, sp2_result_t* ring_entry) {
  if (!refine_active(c)) return;
  __shared__ double sh[8];
  double a = 0.0;
  for (int i = threadIdx.x; i < count; i += 256) a += slots[i];
  a = block_sum(a, sh);
  if (threadIdx.x != 0) return;
  c->tr_d = c->ref_tr; c->tr_dh = a;
  ring_entry->tr_d = c->ref_tr;
  ring_entry->tr_dh = a;
  ring_entry->idem_est = c->ref_tr - c->ref_fro;
  ring_entry->reserved = c->ref_done;
}

}  // namespace

// ------------------------------------------------------------------------------------------
size_t sp2_refine_smem_bytes() { return (size_t)kRStages * 2 * kTileDoubles * sizeof(double); }

cudaError_t sp2_refine_configure() {
  return cudaFuncSetAttribute(k_refine_layer, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sp2_refine_smem_bytes());
}

// enqueue expand + n_layers float64 layers + finalise; returns the number of kernels launched
int sp2_launch_refine(Sp2Ctrl* c, __half* const planes[4] /* Yh0, Ym0, Yh1, Ym1 */, int npad, int N, int n_layers,
                      double* Xa, double* Xb, double* slots, const void* H, sp2_dtype_t in_dt, long ldh,
                      void* D, sp2_dtype_t out_dt, long ldo, sp2_result_t* ring_entry, cudaStream_t s) {
  int launches = 0;
  k_refine_expand<<<npad, 256, 0, s>>>(c, planes[0], planes[1], planes[2], planes[3], npad, Xa, slots); ++launches;
  k_refine_reduce<<<1, 256, 0, s>>>(c, slots, npad); ++launches;
  const int nb = npad / kT;
  const int grid = nb * (nb + 1) / 2;
  double* in = Xa; double* out = Xb;
  for (int r = 0; r < n_layers; ++r) {
    k_refine_layer<<<grid, 256, sp2_refine_smem_bytes(), s>>>(c, in, out, npad, slots, &c->ref_ticket); ++launches;
    double* t = in; in = out; out = t;
  }
#define SP2_RFIN(TI, TO) k_refine_finalise<TI, TO><<<N, 256, 0, s>>>(c, in, npad, (const TI*)H, ldh, (TO*)D, ldo, slots)
  if (in_dt == SP2_F32 && out_dt == SP2_F32) SP2_RFIN(float, float);
  else if (in_dt == SP2_F32 && out_dt == SP2_F64) SP2_RFIN(float, double);
  else if (in_dt == SP2_F64 && out_dt == SP2_F32) SP2_RFIN(double, float);
  else SP2_RFIN(double, double);
#undef SP2_RFIN
  ++launches;
  k_refine_result<<<1, 256, 0, s>>>(c, slots, N, ring_entry); ++launches;
  return launches;
}
