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
//   k_refine_layer     one layer: persistent blocks, 128x128 tiles, producer warp + mbarrier ring, DMMA consumers, fused
//                      update + mirrored store + partials; the last block reduces them and fixes the next branch
//   k_refine_finalise  X -> D in the caller's dtype, tr(DH); result struct
#include <cuda.h>
#include <cuda_runtime.h>
#include <cuda_fp16.h>
#include <stdint.h>
#include "sp2_internal.cuh"
#include "sp2_ptx.cuh"

namespace {

constexpr int kT = 128;          // tile edge
constexpr int kK = 16;           // k doubles per stage
constexpr int kLd = 20;          // padded row pitch of a stage tile in doubles (160 B: 16-B aligned, conflict-free LDS.64)
constexpr int kRStages = 5;
constexpr int kTileDoubles = kT * kLd;

__device__ __forceinline__ void dmma(double& d0, double& d1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0, %1}, {%2}, {%3}, {%0, %1};"
               : "+d"(d0), "+d"(d1)
               : "d"(a), "d"(b));
}

__device__ __forceinline__ double block_sum(double v, double* sh /* one per warp */) {
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
__global__ void __launch_bounds__(256) k_refine_reduce(Sp2Ctrl* c, const double* slots, int count, unsigned int* part_flags,
                                                       int n_flags) {
  for (int i = threadIdx.x; i < n_flags; i += 256) part_flags[i] = 0u;   // the workspace starts with arbitrary contents
  if (!refine_active(c)) return;
  __shared__ double sh[8];
  double a = 0.0, b = 0.0;
  for (int i = threadIdx.x; i < count; i += 256) { a += slots[2 * i]; b += slots[2 * i + 1]; }
  a = block_sum(a, sh);
  b = block_sum(b, sh);
  if (threadIdx.x == 0) refine_decide(c, a, b);
}

// ------------------------------------------------------------------------------------------
// One float64 layer.  Persistent blocks (one per SM) walk the upper-triangular 128x128 tiles in supertiles of
// kRGroup x kRGroup, so that the ~148 tiles in flight share ~2 x kRGroup row panels of X (8 MB each at N = 8192) and stream
// them through L2 together.  Warp-specialised: warp 8 is the producer (one TMA box of 128 rows x kLd doubles per operand
// and k-slice, completion on the stage's `full` mbarrier), warps 0-7 are the DMMA consumers, 2 (rows)
// x 4 (cols), warp tile 64x32 = 8 x 4 DMMA tiles of 8x8 (64 accumulator doubles per thread); they hand a stage back by
// arriving on its `empty` mbarrier.  No block-wide barrier and no per-thread copy instructions in the consumers: the
// first version (every thread issued cp.async, __syncthreads per k-slice) kept the DMMA pipe only 80 % busy, 15 % of the
// warp samples sat at the slice boundary (barrier, and the copies' address registers being recycled).  The ring runs
// on across tile boundaries, so the next tile's operands arrive during this tile's epilogue.
constexpr int kRConsumerWarps = 8;
constexpr int kRThreads = (kRConsumerWarps + 1) * 32;
constexpr int kRGroup = 12;
constexpr int kRMaxBlocks = 256;  // >= SM count of any sm_100 part (flags fit the 1 KB header of the parts region)

// tile t of the grouped order -> (bi, bj), bi <= bj.  Supertiles (I <= J) row-major; inside, rows then columns.
__device__ __forceinline__ void refine_tile(int t, int nb, int& bi, int& bj) {
  const int ng = (nb + kRGroup - 1) / kRGroup;
  for (int I = 0; I < ng; ++I) {
    const int h = min(kRGroup, nb - I * kRGroup);
    for (int J = I; J < ng; ++J) {
      const int w = min(kRGroup, nb - J * kRGroup);
      const int cnt = (I == J) ? h * (h + 1) / 2 : h * w;
      if (t < cnt) {
        int r = 0, cidx = t;
        if (I == J) { while (cidx >= h - r) { cidx -= h - r; ++r; } cidx += r; }
        else { r = t / w; cidx = t - r * w; }
        bi = I * kRGroup + r; bj = J * kRGroup + cidx;
        return;
      }
      t -= cnt;
    }
  }
  bi = bj = 0;   // not reached for t < nb (nb + 1) / 2
}

__global__ void __launch_bounds__(kRThreads, 1) k_refine_layer(Sp2Ctrl* c, const __grid_constant__ CUtensorMap tm_in,
                                                               const double* __restrict__ Xin, double* __restrict__ Xout,
                                                               int npad, double* __restrict__ slots, unsigned int* ticket,
                                                               double* __restrict__ parts, unsigned int* __restrict__ part_flags) {
  if (!refine_active(c)) return;
  extern __shared__ __align__(1024) uint8_t rsm_raw[];
  double* rsm = reinterpret_cast<double*>((reinterpret_cast<uintptr_t>(rsm_raw) + 127) & ~(uintptr_t)127);   // TMA destinations
  __shared__ uint64_t bar_full[kRStages], bar_empty[kRStages];
  const int nb = npad / kT;
  const int n_tiles = nb * (nb + 1) / 2;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const bool plus = c->ref_plus != 0;
  const int KB = npad / kK;
  double tr = 0.0, fro = 0.0;
  // Work split (deterministic): whole tiles round-robin while there are gridDim.x of them left (tile r * grid + b in round
  // r: the blocks of a round share panels and stream them at the same k, which keeps them coincident in L2), then the
  // k-slices of the remaining rem < gridDim.x tiles are cut into gridDim.x equal contiguous ranges, so every block gets
  // the same amount of work whatever the tile count (2080 tiles on 148 SMs otherwise run as 15 rounds of 14.05; the 36
  // tiles of N = 1024 would use 36 SMs).  In that last phase a block whose range starts inside a tile computes that part
  // first and leaves its accumulators in parts[blockIdx.x] (flag set with release); the block whose range starts the
  // tile computes its own part, adds the other blocks' parts in block order and runs the epilogue.
  const int G = (int)gridDim.x;
  const int R = n_tiles / G, rem = n_tiles - R * G;
  const long long rtotal = (long long)rem * KB;
  const long long r_begin = rtotal * blockIdx.x / G, r_end = rtotal * (blockIdx.x + 1) / G;
  // item `it` of this block -> (tile, k-slice range); returns false when the block is done.  rs: cursor of the last phase
  auto next_item = [&](int it, long long& rs, int& t, int& kb_lo, int& kb_hi) -> bool {
    if (it < R) { t = it * G + (int)blockIdx.x; kb_lo = 0; kb_hi = KB; return true; }
    if (rs >= r_end) return false;
    const int tr = (int)(rs / KB);
    kb_lo = (int)(rs - (long long)tr * KB);
    kb_hi = (int)((r_end - (long long)tr * KB) < KB ? (r_end - (long long)tr * KB) : KB);
    t = R * G + tr;
    rs = (long long)tr * KB + kb_hi;
    return true;
  };

  auto stage_a = [&](int s) { return rsm + (size_t)s * 2 * kTileDoubles; };
  auto stage_b = [&](int s) { return rsm + (size_t)s * 2 * kTileDoubles + kTileDoubles; };

  if (tid == 0) {
    for (int s = 0; s < kRStages; ++s) {
      sp2ptx::mbar_init(sp2ptx::smem_u32(&bar_full[s]), 1);
      sp2ptx::mbar_init(sp2ptx::smem_u32(&bar_empty[s]), kRConsumerWarps);
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();

  if (warp == kRConsumerWarps) {
    // ------------------------------------------------ producer (one lane): per k-slice one TMA box per operand,
    // kLd (= kK + 4) doubles wide so that the rows land in shared memory with the padded pitch the fragment loads want
    if (sp2ptx::elect_one()) {
      int stage = 0; uint32_t phase = 0;
      long long rs = r_begin;
      int t, kb_lo, kb_hi;
      for (int it = 0; next_item(it, rs, t, kb_lo, kb_hi); ++it) {
        int bi, bj;
        refine_tile(t, nb, bi, bj);
        for (int kb = kb_lo; kb < kb_hi; ++kb) {
          sp2ptx::mbar_wait(sp2ptx::smem_u32(&bar_empty[stage]), phase ^ 1u);
          const uint32_t full = sp2ptx::smem_u32(&bar_full[stage]);
          sp2ptx::mbar_expect_tx(full, 2u * kTileDoubles * (uint32_t)sizeof(double));
          sp2ptx::tma_load_2d<1>(sp2ptx::smem_u32(stage_a(stage)), &tm_in, full, kb * kK, bi * kT);
          sp2ptx::tma_load_2d<1>(sp2ptx::smem_u32(stage_b(stage)), &tm_in, full, kb * kK, bj * kT);
          if (++stage == kRStages) { stage = 0; phase ^= 1u; }
        }
      }
    }
  } else {
    // ------------------------------------------------ DMMA consumers
    const int wm = warp >> 2, wn = warp & 3;                 // 2 x 4 warps
    const int g = lane >> 2, q = lane & 3;                   // DMMA fragment coordinates
    int stage = 0; uint32_t phase = 0;
    long long rs = r_begin;
    int t, kb_lo, kb_hi;
    for (int it = 0; next_item(it, rs, t, kb_lo, kb_hi); ++it) {
      int bi, bj;
      refine_tile(t, nb, bi, bj);
      const int i0 = bi * kT, j0 = bj * kT;
      double acc[8][4][2];
#pragma unroll
      for (int a = 0; a < 8; ++a)
#pragma unroll
        for (int b = 0; b < 4; ++b) { acc[a][b][0] = 0.0; acc[a][b][1] = 0.0; }

      for (int kb = kb_lo; kb < kb_hi; ++kb) {
        sp2ptx::mbar_wait(sp2ptx::smem_u32(&bar_full[stage]), phase);
        const double* A = stage_a(stage) + (wm * 64 + g) * kLd + q;
        const double* B = stage_b(stage) + (wn * 32 + g) * kLd + q;
#pragma unroll
        for (int k4 = 0; k4 < kK / 4; ++k4) {
          double af[8], bf[4];
#pragma unroll
          for (int a = 0; a < 8; ++a) af[a] = A[a * 8 * kLd + k4 * 4];
#pragma unroll
          for (int b = 0; b < 4; ++b) bf[b] = B[b * 8 * kLd + k4 * 4];
#pragma unroll
          for (int a = 0; a < 8; ++a)
#pragma unroll
            for (int b = 0; b < 4; ++b) dmma(acc[a][b][0], acc[a][b][1], af[a], bf[b]);
        }
        __syncwarp();
        if (lane == 0) sp2ptx::mbar_arrive(sp2ptx::smem_u32(&bar_empty[stage]));
        if (++stage == kRStages) { stage = 0; phase ^= 1u; }
      }

      if (kb_lo > 0) {
        // a later part of a tile that another block started: park the accumulators (thread-private order, coalesced)
        double* mine = parts + (size_t)blockIdx.x * (kT * kT) + tid;
#pragma unroll
        for (int a = 0; a < 8; ++a)
#pragma unroll
          for (int b = 0; b < 4; ++b) {
            __stcg(mine + (size_t)((a * 4 + b) * 2 + 0) * (kRConsumerWarps * 32), acc[a][b][0]);
            __stcg(mine + (size_t)((a * 4 + b) * 2 + 1) * (kRConsumerWarps * 32), acc[a][b][1]);
          }
        __threadfence();
        asm volatile("bar.sync 1, %0;" ::"n"(kRConsumerWarps * 32) : "memory");
        if (tid == 0) asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(part_flags + blockIdx.x), "r"(1u) : "memory");
        continue;
      }
      if (kb_hi < KB) {
        // this block started the tile: add the parts of the blocks that continue it, in block order
        for (int j = blockIdx.x + 1; j < G && rtotal * j / G < (long long)(t - R * G + 1) * KB; ++j) {
          if (tid == 0) {
            unsigned int v = 0;
            long long spins = 0;
            do {
              asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(part_flags + j) : "memory");
              if (++spins > sp2ptx::kSpinLimit) __trap();
            } while (v == 0u);
          }
          asm volatile("bar.sync 1, %0;" ::"n"(kRConsumerWarps * 32) : "memory");
          const double* theirs = parts + (size_t)j * (kT * kT) + tid;
#pragma unroll
          for (int a = 0; a < 8; ++a)
#pragma unroll
            for (int b = 0; b < 4; ++b) {
              acc[a][b][0] += __ldcg(theirs + (size_t)((a * 4 + b) * 2 + 0) * (kRConsumerWarps * 32));
              acc[a][b][1] += __ldcg(theirs + (size_t)((a * 4 + b) * 2 + 1) * (kRConsumerWarps * 32));
            }
        }
      }

      // epilogue: X' = X^2 or 2X - X^2; elements with gj >= gi only, mirrored; partials
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
    }
  }

  __shared__ double sh[kRThreads / 32];
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
  for (int i = tid; i < (int)gridDim.x; i += kRThreads) { a += __ldcg(slots + 2 * i); b += __ldcg(slots + 2 * i + 1); }
  a = block_sum(a, sh);
  b = block_sum(b, sh);
  for (int i = tid; i < (int)gridDim.x; i += kRThreads) part_flags[i] = 0u;     // every part was consumed
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
size_t sp2_refine_smem_bytes() { return (size_t)kRStages * 2 * kTileDoubles * sizeof(double) + 1024; }
// TMA box of the float64 iterates: {k extent, rows} in doubles
void sp2_refine_box(int* box_k, int* box_rows) { *box_k = kLd; *box_rows = kT; }

static int refine_sm_count() {
  int dev = 0, sms = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms < 1)
    sms = 148;
  return sms;
}

cudaError_t sp2_refine_configure() {
  return cudaFuncSetAttribute(k_refine_layer, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sp2_refine_smem_bytes());
}

// enqueue expand + n_layers float64 layers + finalise; returns the number of kernels launched
// scratch of the split tiles: one flag and one 128x128 accumulator image per block
int sp2_refine_max_blocks() { return kRMaxBlocks; }
size_t sp2_refine_parts_bytes(int blocks) { return 1024 + (size_t)blocks * kT * kT * sizeof(double); }
int sp2_refine_grid(int npad, int max_blocks) {
  const int nb = npad / kT;
  const long long total = (long long)(nb * (nb + 1) / 2) * (npad / kK);   // k-slices of a layer
  int grid = refine_sm_count();
  if (max_blocks > 0 && grid > max_blocks) grid = max_blocks;
  if (grid > kRMaxBlocks) grid = kRMaxBlocks;
  if ((long long)grid * 4 > total) grid = (int)(total / 4);           // at least four k-slices per block
  return grid < 1 ? 1 : grid;
}

// enqueue expand + n_layers float64 layers + finalise; returns the number of kernels launched.  The blocks of a layer
// hand partial tiles to one another (see k_refine_layer), so its grid (sp2_refine_grid) must be co-resident: one block per
// SM, at most max_blocks of them (sp2_options_t.max_ctas).
int sp2_launch_refine(Sp2Ctrl* c, __half* const planes[4] /* Yh0, Ym0, Yh1, Ym1 */, int npad, int N, int n_layers,
                      double* Xa, double* Xb, const CUtensorMap* maps /* of Xa, Xb: sp2_refine_box() */, double* slots,
                      void* parts_region, int max_blocks, const void* H, sp2_dtype_t in_dt, long ldh,
                      void* D, sp2_dtype_t out_dt, long ldo, sp2_result_t* ring_entry, cudaStream_t s) {
  int launches = 0;
  unsigned int* part_flags = static_cast<unsigned int*>(parts_region);
  double* parts = reinterpret_cast<double*>(static_cast<uint8_t*>(parts_region) + 1024);
  const int grid = sp2_refine_grid(npad, max_blocks);
  k_refine_expand<<<npad, 256, 0, s>>>(c, planes[0], planes[1], planes[2], planes[3], npad, Xa, slots); ++launches;
  k_refine_reduce<<<1, 256, 0, s>>>(c, slots, npad, part_flags, grid); ++launches;
  double* in = Xa; double* out = Xb;
  for (int r = 0; r < n_layers; ++r) {
    k_refine_layer<<<grid, kRThreads, sp2_refine_smem_bytes(), s>>>(c, maps[r & 1], in, out, npad, slots, &c->ref_ticket, parts,
                                                                     part_flags); ++launches;
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
