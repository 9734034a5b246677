// sp2_layer.cu -- one DNN-SP2 layer as a persistent, warp-specialised
// sm_100a kernel: TMA -> shared-memory ring -> tcgen05.mma (FP16 x FP16 -> FP32 in TMEM) -> fused
// epilogue (update, hi/lo split, mirrored store, trace partials) -> last CTA runs the controller.
//
// What a layer computes: X_{n+1} = X_n^2 or 2X_n - X_n^2.  With the shifted
// iterate X = c I + Y this is Y' = alpha*Y + sigma*Y^2 and, for the first-order iterate,
// Z' = alpha*Z + sigma*(YZ + ZY).  With the dual half-precision representation of PAPER.md:153-170
// (Eq. 20-22)  Y = h + m, Z = p + q  the products are
//     Y^2     ~ h h + h m + m h                                   (m m dropped, Eq. 22)
//     YZ + ZY ~ (h p + h q + m p) + (p h + p m + q h)
// All planes are symmetric, so B[k][j] = B[j][k] and both operands of every product are K-major
// row panels of the same row-major plane; only tiles on or above the diagonal are computed and
// every result is written to (i,j) and (j,i), which keeps the planes bit-symmetric.
//
// A work unit = one output tile of one product class, expressed as `passes` sweeps over k of
//     acc += A0 B0^T + A0 B1^T + A1 B0^T
// (Y^2: one pass with A=(h,m) rows i, B=(h,m) rows j;  YZ+ZY: pass 0 A=(h,m), B=(p,q); pass 1
// A=(p,q), B=(h,m)).
//
// CG = 1: tile 128x128, one CTA, UMMA 128x128x16.  CG = 2: tile 256x256 on a CTA pair
// (cta_group::2, UMMA 256x256x16); each CTA loads 128 rows of A and 128 rows of B per plane.
#include <cuda.h>
#include "sp2_internal.cuh"
#include "sp2_layer.h"
#include "sp2_ptx.cuh"

namespace {

// Shared-memory ring: 3 stages of 64 k-elements (64 KB: A.hi, A.lo, B.hi, B.lo boxes with 128-byte rows,
// SWIZZLE_128B).  7 stages of 32 k-elements (32 KB, SWIZZLE_64B; kBK = 32, kStages = 7 also builds) keep more
// bytes in flight but measured the same speed with 10 % more DRAM traffic, so the coarser ring stays.
constexpr int kBK = 64;                       // k elements per stage
constexpr int kRows = 128;                    // rows per TMA box / per CTA operand tile
constexpr int kStages = 3;
constexpr int kPlaneTileBytes = kRows * kBK * 2;          // 16 KB
constexpr int kStageBytes = 4 * kPlaneTileBytes;          // A0, A1, B0, B1 = 64 KB
constexpr int kSwizzleBytes = kBK * 2;                    // swizzle span = one row of the box
static_assert(kBK == 32 || kBK == 64, "box rows are 64 or 128 bytes");
constexpr int kThreads = 384;                 // 4 producer-side warps + 8 consumer warps
constexpr int kConsumerWarps = 8;              // warps 0..7
// The issue arbiter favours high warp ids, so the latency-critical single-thread roles sit above the consumers
// (measured neutral at N = 8192; kept because it cannot hurt).
constexpr int kWarpTma = 8, kWarpMma = 9, kWarpAlloc = 10;
constexpr int kRegsProducer = 40;             // setmaxnreg budgets: 128*40 + 256*232 <= 65536
constexpr int kRegsConsumer = 232;

using namespace sp2ptx;
__device__ __forceinline__ uint64_t make_smem_desc(uint32_t saddr) { return make_smem_desc_sw<kSwizzleBytes>(saddr); }

struct alignas(8) SmemBarriers {
  uint64_t full[kStages];
  uint64_t empty[kStages];
  uint64_t tmem_full[2];
  uint64_t tmem_empty[2];
  uint32_t tmem_base;
  uint32_t is_last;
  // persistent mode: stop = the consumers saw the controller's done flag; prod_layers = layers the TMA producer has
  // started; prod_final = it will start no more (the MMA issuer follows the producer)
  uint32_t stop, prod_layers, prod_final, pad0;
  double red[32];         // persistent mode: warp partials of the slot reduction
  // persistent mode: this CTA's own copy of the control block (every CTA runs the controller, see persist_control)
  alignas(8) uint8_t ctrl_copy[sizeof(Sp2Ctrl)];
  // 32x32 diagonal blocks in flight, one per TMEM lane quarter (of the two warps of a quarter only one holds the
  // diagonal): packed hi | lo << 16 per element, rows padded to 33 words (conflict-free row and column reads)
  uint32_t diag_t[4][32 * 33];
  // partial sums of this CTA, per consumer warp and product class (0: Y^2, 1 + b: Y Z_b + Z_b Y): one writer each
  // (lane 0 of the warp), reduced in fixed order at the end of the kernel into ONE slot per CTA and class
  Sp2Slot acc[kConsumerWarps][1 + SP2_NB];
};

// (.cg: L2 only.  In the persistent mode other CTAs rewrite these planes between layers of the SAME kernel, so a line
// left in this SM's L1 by an earlier layer would be stale; the reads have no L1 reuse anyway.)
__device__ __forceinline__ uint4 ld_global_v4(const void* p) {
  uint4 r;
  asm volatile("ld.global.cg.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p));
  return r;
}

// streaming (evict-first) stores: the new planes are not re-read in this launch and must not push the
// operand panels out of L2
__device__ __forceinline__ void st_cs_v4(void* p, uint32_t a, uint32_t b, uint32_t c, uint32_t d) {
  asm volatile("st.global.cs.v4.u32 [%0], {%1, %2, %3, %4};" ::"l"(p), "r"(a), "r"(b), "r"(c), "r"(d) : "memory");
}
__device__ __forceinline__ void st_cs_u16(void* p, uint32_t v) {
  asm volatile("st.global.cs.u16 [%0], %1;" ::"l"(p), "h"((unsigned short)v) : "memory");
}

__device__ __forceinline__ uint32_t u4_word(const uint4& v, int i) {
  return i == 0 ? v.x : (i == 1 ? v.y : (i == 2 ? v.z : v.w));
}

// The scalar part of a layer boundary in one thread: trace identity, rescaled sums, controller.  Not inlined: its
// float64 code (a batch of loads, arithmetic in registers, a batch of stores) must not add to the register pressure
// of the kernels around it.
__device__ __noinline__ void layer_scalar_control(Sp2Ctrl* ctrl, double tr, double fro, double mx, double tracc) {
  sp2_trace_identity(ctrl, tracc);
  const double sy = sp2_exp2i(-ctrl->t);
  ctrl->tr_y = tr * sy; ctrl->fro_y = fro * sy * sy; ctrl->max_y = mx * sy;
  sp2_controller(ctrl);
}

// ----------------------------------------------------------------------------------------------
// shared tail of both engines: last block reduces the slots (index order) and runs the controller
// slot array: [z slots of perturbation 0 (n_z)] ... [z slots of perturbation nb - 1][y slots (n_y)]
__device__ inline void layer_tail(Sp2Ctrl* ctrl, const Sp2Slot* slots, int n_y, int n_z, int nb,
                                  unsigned int n_blocks, uint32_t* is_last_smem, double* red,
                                  unsigned int* flags = nullptr, int n_flags = 0) {
  __syncthreads();
  if (threadIdx.x == 0) {
    __threadfence();
    const unsigned int old = atomicAdd(&ctrl->ticket, 1u);
    *is_last_smem = (old == n_blocks - 1) ? 1u : 0u;
  }
  __syncthreads();
  if (!*is_last_smem) return;
  __threadfence();
  for (int i = threadIdx.x; i < n_flags; i += blockDim.x) flags[i] = 0u;   // every split unit was consumed (and the lockstep counters)
  double tr, fro, mx, tracc, unused;
  sp2_reduce_slots(slots + (size_t)nb * n_z, n_y, red, tr, fro, mx, tracc);
  for (int b = 0; b < nb; ++b) {
    double trz, froz, mxz;
    sp2_reduce_slots(slots + (size_t)b * n_z, n_z, red, trz, froz, mxz, unused);
    if (threadIdx.x == 0) {
      const double sz = sp2_exp2i(-ctrl->u[b]);
      ctrl->tr_z[b] = trz * sz; ctrl->fro_z[b] = froz * sz * sz; ctrl->max_z[b] = mxz * sz;
    }
  }
  if (threadIdx.x == 0) {
    ctrl->ticket = 0;
    layer_scalar_control(ctrl, tr, fro, mx, tracc);
  }
}

// ----------------------------------------------------------------------------------------------
// Epilogue of one 32-column chunk held in registers (acc[0..31] = FP32 sums of row gi, columns
// gj0..gj0+31): update, split, mirrored store, partial sums.
struct EpiPartials { double tr, fro, tracc; float mx; };

// Old-tile prefetch buffer of the epilogue: the hi and lo words of one 32-column chunk of this
// thread's row (4 + 4 uint4 = 32 registers), refilled one chunk ahead while the current chunk is
// processed, so the epilogue is never stalled on a global-load round trip.
struct EpiOld { uint4 h[4], m[4]; };

__device__ __forceinline__ void epilogue_prefetch(EpiOld& o, int gi, int gj0, size_t npad,
                                                  const __half* __restrict__ in_h, const __half* __restrict__ in_m) {
  const uint4* ph = reinterpret_cast<const uint4*>(in_h + (size_t)gi * npad + gj0);
  const uint4* pm = reinterpret_cast<const uint4*>(in_m + (size_t)gi * npad + gj0);
#pragma unroll
  for (int w = 0; w < 4; ++w) { o.h[w] = ld_global_v4(ph + w); o.m[w] = ld_global_v4(pm + w); }
}

__device__ __forceinline__ float2 h2_to_f2(uint32_t w) {
  return __half22float2(*reinterpret_cast<const __half2*>(&w));
}
__device__ __forceinline__ uint32_t f2_to_h2(float a, float b) {
  const __half2 h = __floats2half2_rn(a, b);
  return *reinterpret_cast<const uint32_t*>(&h);
}

// One 32-column chunk that lies entirely above the diagonal (the common case: no diagonal element, every element
// counts twice in ||.||_F^2 and is stored twice).  The statistics use the FP32 value before the split (it differs
// from the stored hi+lo by an unbiased 2^-22 relative rounding; a non-finite value still reaches the controller
// through the Frobenius sum).
__device__ __forceinline__ void epilogue_chunk_full(const float* acc, EpiOld& old, const uint4* next_h, const uint4* next_m,
                                                    int gi, int gj0,
                                                    size_t npad, __half* __restrict__ out_h, __half* __restrict__ out_m,
                                                    float a1hi, float a1lo, float a2,
                                                    uint32_t lo_round, uint32_t lo_mask, EpiPartials& P) {
  unsigned short* th = reinterpret_cast<unsigned short*>(out_h) + (size_t)gj0 * npad + gi;   // mirrored image
  unsigned short* tm = reinterpret_cast<unsigned short*>(out_m) + (size_t)gj0 * npad + gi;
  float fsum = 0.f, mx = P.mx;
#pragma unroll
  for (int w = 0; w < 4; ++w) {               // 8 columns at a time keeps the live register set small
    uint32_t nh[4], nm[4];                    // packed pairs of new hi / lo halves
    const uint4 oh = old.h[w], om = old.m[w];
    if (next_h) { old.h[w] = ld_global_v4(next_h + w); old.m[w] = ld_global_v4(next_m + w); }   // one chunk ahead
#pragma unroll
    for (int pr = 0; pr < 4; ++pr) {
      const float2 fh = h2_to_f2(u4_word(oh, pr)), fm = h2_to_f2(u4_word(om, pr));
      const float old0 = fh.x + fm.x, old1 = fh.y + fm.y;
      const int ci = 8 * w + 2 * pr;
      const float y0 = fmaf(a1hi, old0, fmaf(a1lo, old0, a2 * acc[ci]));
      const float y1 = fmaf(a1hi, old1, fmaf(a1lo, old1, a2 * acc[ci + 1]));
      nh[pr] = f2_to_h2(y0, y1);
      const float2 hb = h2_to_f2(nh[pr]);
      nm[pr] = (f2_to_h2(y0 - hb.x, y1 - hb.y) + lo_round) & lo_mask;   // lo_mask = ~0: all 11 bits of the lo plane
      fsum = fmaf(y0, y0, fsum);
      fsum = fmaf(y1, y1, fsum);
      mx = fmaxf(mx, fmaxf(fabsf(y0), fabsf(y1)));
    }
    st_cs_v4(out_h + (size_t)gi * npad + gj0 + 8 * w, nh[0], nh[1], nh[2], nh[3]);
    st_cs_v4(out_m + (size_t)gi * npad + gj0 + 8 * w, nm[0], nm[1], nm[2], nm[3]);
#pragma unroll
    for (int pr = 0; pr < 4; ++pr) {        // lanes = consecutive rows -> 64 contiguous bytes per warp store
      st_cs_u16(th, nh[pr] & 0xffffu);
      st_cs_u16(tm, nm[pr] & 0xffffu);
      st_cs_u16(th + npad, nh[pr] >> 16);
      st_cs_u16(tm + npad, nm[pr] >> 16);
      th += 2 * npad; tm += 2 * npad;
    }
  }
  P.mx = mx;
  P.fro += (double)(2.f * fsum);
}

// The 32-column chunk that holds the diagonal: the 32 x 32 block rows gj0 .. gj0 + 31 (one row per lane) by the same
// columns.  Only elements on or above the diagonal are COMPUTED (hi*lo and lo*hi cross terms add in a different order
// for (i,j) and (j,i), so the two accumulators may differ in the last bit); they go through a shared-memory tile, and
// every lane then assembles its whole row -- its own values right of the diagonal, the other lanes' values left of
// it -- and stores it with 16-byte vectors: the block is bit-symmetric by construction and no store is narrower than
// 16 bytes (element-wise 2-byte stores, 32 rows apart per lane, made this chunk cost 8 us: the floor of small N).
// T: this warp's tile (32 x 33 words, hi | lo << 16).  The statistics use the exact stored values.
__device__ __forceinline__ void epilogue_chunk_diag(const float* acc, EpiOld& old, const uint4* next_h, const uint4* next_m,
                                                    int gi, int gj0,
                                                    size_t npad, __half* __restrict__ out_h, __half* __restrict__ out_m,
                                                    float a1hi, float a1lo, float a2, float dsh_hi, float dsh_lo,
                                                    uint32_t lo_round, uint32_t lo_mask, uint32_t* __restrict__ T, EpiPartials& P) {
  const int r = gi - gj0;                     // row inside the block = lane
  uint32_t* Trow = T + r * 33;
  float dacc = 0.f, dval = 0.f;               // this row's diagonal accumulator and stored diagonal value
#pragma unroll
  for (int w = 0; w < 4; ++w) {
    const uint4 oh = old.h[w], om = old.m[w];
    if (next_h) { old.h[w] = ld_global_v4(next_h + w); old.m[w] = ld_global_v4(next_m + w); }   // one chunk ahead
#pragma unroll
    for (int pr = 0; pr < 4; ++pr) {
      const float2 fh = h2_to_f2(u4_word(oh, pr)), fm = h2_to_f2(u4_word(om, pr));
      const float old0 = fh.x + fm.x, old1 = fh.y + fm.y;
      const int ci = 8 * w + 2 * pr;
      float y0 = fmaf(a1hi, old0, fmaf(a1lo, old0, a2 * acc[ci]));
      float y1 = fmaf(a1hi, old1, fmaf(a1lo, old1, a2 * acc[ci + 1]));
      if (ci == r) { y0 = (y0 + dsh_lo) + dsh_hi; dacc = acc[ci]; }
      if (ci + 1 == r) { y1 = (y1 + dsh_lo) + dsh_hi; dacc = acc[ci + 1]; }
      const uint32_t nh = f2_to_h2(y0, y1);
      const float2 hb = h2_to_f2(nh);
      const uint32_t nm = (f2_to_h2(y0 - hb.x, y1 - hb.y) + lo_round) & lo_mask;
      Trow[ci] = (nh & 0xffffu) | (nm << 16);
      Trow[ci + 1] = (nh >> 16) | (nm & 0xffff0000u);
    }
  }
  __syncwarp();
  float fsum = 0.f, mx = P.mx;
#pragma unroll
  for (int w = 0; w < 4; ++w) {
    uint32_t nh[4], nm[4];
#pragma unroll
    for (int pr = 0; pr < 4; ++pr) {
      const int c0 = 8 * w + 2 * pr, c1 = c0 + 1;
      const uint32_t e0 = T[(c0 >= r) ? r * 33 + c0 : c0 * 33 + r];  // left of the diagonal: the mirror image
      const uint32_t e1 = T[(c1 >= r) ? r * 33 + c1 : c1 * 33 + r];
      nh[pr] = (e0 & 0xffffu) | (e1 << 16);
      nm[pr] = (e0 >> 16) | (e1 & 0xffff0000u);
      const float2 hv = h2_to_f2(nh[pr]), mv = h2_to_f2(nm[pr]);
      const float s0 = hv.x + mv.x, s1 = hv.y + mv.y;
      fsum = fmaf(s0, s0, fsum);              // the whole symmetric row: off-diagonal elements of the block count twice
      fsum = fmaf(s1, s1, fsum);
      mx = fmaxf(mx, fmaxf(fabsf(s0), fabsf(s1)));
      if (c0 == r) dval = s0;
      if (c1 == r) dval = s1;
    }
    st_cs_v4(out_h + (size_t)gi * npad + gj0 + 8 * w, nh[0], nh[1], nh[2], nh[3]);
    st_cs_v4(out_m + (size_t)gi * npad + gj0 + 8 * w, nm[0], nm[1], nm[2], nm[3]);
  }
  __syncwarp();                               // the tile is free for this warp's next diagonal block
  P.mx = mx;
  P.fro += (double)fsum;
  P.tr += (double)dval;
  P.tracc += (double)dacc;
}

// Fused epilogue of this thread's row over NCH chunks of 32 columns held in registers
// (acc[0 .. 32 NCH) = FP32 sums of row gi, columns j0 ..): update, split, mirrored store, partial sums.
// `old` holds chunk 0 on entry and is refilled one chunk ahead.
template <int NCH>
__device__ __forceinline__ void epilogue_row(const float* acc, EpiOld& old, int gi, int j0, size_t npad,
                                             const __half* __restrict__ in_h, const __half* __restrict__ in_m,
                                             __half* __restrict__ out_h, __half* __restrict__ out_m,
                                             float a1hi, float a1lo, float a2, float dsh_hi, float dsh_lo,
                                             uint32_t lo_round, uint32_t lo_mask, uint32_t* __restrict__ T, EpiPartials& P) {
#pragma unroll
  for (int ch = 0; ch < NCH; ++ch) {
    const int gj0 = j0 + ch * 32;
    const uint4* nxh = (ch + 1 < NCH) ? reinterpret_cast<const uint4*>(in_h + (size_t)gi * npad + gj0 + 32) : nullptr;
    const uint4* nxm = (ch + 1 < NCH) ? reinterpret_cast<const uint4*>(in_m + (size_t)gi * npad + gj0 + 32) : nullptr;
    // gi = 32-aligned base + lane and gj0 is 32-aligned, so both tests are warp-uniform
    if (gj0 > gi) {                           // entirely above the diagonal
      epilogue_chunk_full(&acc[ch * 32], old, nxh, nxm, gi, gj0, npad, out_h, out_m, a1hi, a1lo, a2, lo_round, lo_mask, P);
    } else if (gj0 + 31 >= gi) {              // holds the diagonal
      epilogue_chunk_diag(&acc[ch * 32], old, nxh, nxm, gi, gj0, npad, out_h, out_m, a1hi, a1lo, a2, dsh_hi, dsh_lo,
                          lo_round, lo_mask, T, P);
    } else if (nxh) {                         // entirely below: mirrored by its transpose; keep the prefetch rolling
      epilogue_prefetch(old, gi, gj0 + 32, npad, in_h, in_m);
    }
  }
}

// Epilogue of the plain-product mode: this thread's row gi, columns j0 .. j0 + COLS of C = A B^T.
//   out_kind 0: hi/lo FP16 planes at the exponent folded into `scale` (feeds the next product)
//   out_kind 1 / 2: the caller's float / double matrix (rows and columns < n only)
template <int COLS>
__device__ __forceinline__ void gemm_epilogue(const float* acc, int gi, int j0, const Sp2LayerArgs& a, double scale) {
  if (a.out_kind == 0) {
    const float sc = (float)scale;
    __half* ph = a.out[0] + (size_t)gi * a.npad + j0;
    __half* pm = a.out[1] + (size_t)gi * a.npad + j0;
#pragma unroll
    for (int w = 0; w < COLS / 8; ++w) {
      uint32_t nh[4], nm[4];
#pragma unroll
      for (int pr = 0; pr < 4; ++pr) {
        const float y0 = acc[8 * w + 2 * pr] * sc, y1 = acc[8 * w + 2 * pr + 1] * sc;
        nh[pr] = f2_to_h2(y0, y1);
        const float2 hb = h2_to_f2(nh[pr]);
        nm[pr] = f2_to_h2(y0 - hb.x, y1 - hb.y);
      }
      *reinterpret_cast<uint4*>(ph + 8 * w) = make_uint4(nh[0], nh[1], nh[2], nh[3]);
      *reinterpret_cast<uint4*>(pm + 8 * w) = make_uint4(nm[0], nm[1], nm[2], nm[3]);
    }
    return;
  }
  if (gi >= a.n) return;
  if (a.out_kind == 2) {
    double* c = reinterpret_cast<double*>(a.cout) + (size_t)gi * a.ldc;
#pragma unroll
    for (int k = 0; k < COLS; ++k) if (j0 + k < a.n) c[j0 + k] = (double)acc[k] * scale;
  } else {
    float* c = reinterpret_cast<float*>(a.cout) + (size_t)gi * a.ldc;
    const float sc = (float)scale;
#pragma unroll
    for (int k = 0; k < COLS; ++k) if (j0 + k < a.n) c[j0 + k] = acc[k] * sc;
  }
}

// ----------------------------------------------------------------------------------------------
// Persistent multi-layer mode (small and medium N, where a layer is shorter than a kernel launch and its tail):
// ONE launch runs the whole stack.  Between layers the CTAs meet at a grid-wide barrier (every CTA of the grid is
// resident: the grid is bounded by the co-residency query of sp2_create) that has two halves:
//   arrive   each CTA stores its planes and its partial sums and takes a ticket (a counter that only grows);
//   release  the CTA that draws the last ticket of the layer reduces the slots, runs the controller for the next
//            layer and publishes the new epoch; the consumer warps of every CTA wait for that epoch.
// The MMAs of layer n + 1 need the planes of layer n but NOT the controller's decision (branch and coefficients only
// enter the epilogue), so the TMA producer waits for the arrive half alone (ticket count) and the tensor core runs
// layer n + 1 while the controller of layer n is still at work.  When the controller says stop, that one layer has
// been started in vain: the consumers drain its accumulators without an epilogue.  Barriers, TMEM and the pipeline
// phases live across layers; the ping-pong planes swap by layer parity (both argument blocks live in global memory).
__device__ __forceinline__ void named_bar_sync(int id, int nthreads) {
  asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}
// generic-proxy global writes of this thread -> visible to later async-proxy (TMA) reads
__device__ __forceinline__ void fence_proxy_async_global() { asm volatile("fence.proxy.async.global;" ::: "memory"); }

__device__ __forceinline__ unsigned int ld_acquire_u32(const unsigned int* p) {
  unsigned int v;
  asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ void st_release_u32(unsigned int* p, unsigned int v) {
  asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}

// Reduce the per-CTA slots of one class with the 256 consumer threads (count <= 256): one slot per thread, fixed
// shuffle tree, eight warp partials added in index order by thread 0.  Deterministic.  Result valid in thread 0.
__device__ __forceinline__ void reduce_slots_fast(const Sp2Slot* slots, int count, double* red /* smem 4 x 8 */,
                                                  double& tr, double& fro, double& mx, double& tracc) {
  const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
  double a = 0.0, b = 0.0, d = 0.0, m = 0.0;
  if (tid < count) {         // past L1: written by other CTAs of this kernel
    a = __ldcg(&slots[tid].tr); b = __ldcg(&slots[tid].fro); d = __ldcg(&slots[tid].tracc); m = (double)__ldcg(&slots[tid].mx);
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    a += __shfl_xor_sync(0xffffffffu, a, o);
    b += __shfl_xor_sync(0xffffffffu, b, o);
    d += __shfl_xor_sync(0xffffffffu, d, o);
    const double q = __shfl_xor_sync(0xffffffffu, m, o);
    m = (q > m || q != q) ? q : m;
  }
  if (lane == 0) { red[w] = a; red[8 + w] = b; red[16 + w] = d; red[24 + w] = m; }
  named_bar_sync(1, kConsumerWarps * 32);
  if (tid == 0) {
    a = red[0]; b = red[8]; d = red[16]; m = red[24];
    for (int k = 1; k < kConsumerWarps; ++k) {
      a += red[k]; b += red[8 + k]; d += red[16 + k];
      const double q = red[24 + k];
      m = (q > m || q != q) ? q : m;
    }
    tr = a; fro = b; tracc = d; mx = m;
  }
  named_bar_sync(1, kConsumerWarps * 32);
}

// Persistent mode, after the grid barrier of a layer (every CTA has drawn its ticket): the controller, REPLICATED.
// Every CTA reduces the per-CTA slots of the layer in the same fixed order and runs the same scalar controller on its own
// shared-memory copy of the control block, so all of them hold the same coefficients, branch and stop decision without
// a second, release half of the barrier (one CTA computing, writing back, fencing, releasing, everybody else polling and
// re-reading: 5 us of the ~9 us that serial tail took per layer).  Block 0 alone writes the history entries to global
// memory.  Not inlined: its double-precision scalar code must not add to the register pressure of the layer loop.
__device__ __noinline__ void persist_control(const Sp2LayerArgs& a, SmemBarriers* bars, const Sp2Slot* slots, int nb, int nblk) {
  Sp2Ctrl* ctrl = reinterpret_cast<Sp2Ctrl*>(bars->ctrl_copy);
  double* redf = reinterpret_cast<double*>(bars->red);
  double tr, fro, mx, tracc, unused;
  reduce_slots_fast(slots + (size_t)nb * nblk, nblk, redf, tr, fro, mx, tracc);
  for (int b = 0; b < nb; ++b) {
    double trz, froz, mxz;
    reduce_slots_fast(slots + (size_t)b * nblk, nblk, redf, trz, froz, mxz, unused);
    if (threadIdx.x == 0) {
      const double sz = sp2_exp2i(-ctrl->u[b]);
      ctrl->tr_z[b] = trz * sz; ctrl->fro_z[b] = froz * sz * sz; ctrl->max_z[b] = mxz * sz;
    }
  }
  if (threadIdx.x == 0) {
    const int n = ctrl->n;                   // the controller reads e[n - 2] and writes tr_x[n], e[n] (local history)
    layer_scalar_control(ctrl, tr, fro, mx, tracc);
    if (blockIdx.x == 0 && n < SP2_LAYER_CAP) { a.ctrl->tr_x[n] = ctrl->tr_x[n]; a.ctrl->e[n] = ctrl->e[n]; }
  }
  named_bar_sync(1, kConsumerWarps * 32);
}

// ----------------------------------------------------------------------------------------------
// Warp roles (384 threads): warps 0..7 consumers; warp 8 TMA producer, warp 9 MMA issuer, warp 10 TMEM
// allocator, warp 11 idle.  The k range of a unit is cut into segments of seg_kb k-blocks; each
// segment is accumulated by the tensor core into a fresh TMEM buffer (2 buffers, ping-pong) and
// the consumers add the finished segment into FP32 register sums with round-to-nearest adds.
// This bounds the length of the truncating in-TMEM accumulation (DESIGN.md "Tensor-core
// truncation bias") and costs no tensor time: the drain overlaps the next segment's MMAs.
// MODE 0: one SP2 layer.  MODE 1: the same mainloop as a plain product C = A B^T of two hi/lo plane pairs (A = tm[0..1],
// B = tm[2..3]; every tile, no mirror, no controller) for the congruence transforms of sp2_congruence.
// PERSIST: the whole layer stack in one launch (see above); args[0] reads buffer 0 and writes buffer 1, args[1] the reverse.
template <int CG, int MODE, bool PERSIST>
__device__ __forceinline__ void layer_body(const Sp2LayerArgs* __restrict__ args) {
  constexpr int TILE = 128 * CG;          // output tile edge
  constexpr int UM = 128 * CG, UN = 128 * CG;
  constexpr int ACC_COLS = UN;            // FP32 accumulator columns per TMEM buffer
  constexpr int WCOLS = ACC_COLS / 2;     // columns per consumer warp (two warps per TMEM lane quarter)
  constexpr int NCH = WCOLS / 32;         // 32-column chunks per consumer warp
  constexpr uint32_t TMEM_COLS = 2 * ACC_COLS;
  constexpr uint32_t IDESC = make_idesc(UM, UN);
  static_assert(!(PERSIST && MODE == 1), "the plain-product mode is a single launch");

  // Programmatic dependent launch: let the next layer's CTAs be scheduled as soon as SMs free up; everything
  // up to griddepcontrol.wait below (barrier init, TMEM allocation, work-list offsets) then overlaps the tail
  // of the previous layer.  Nothing the previous launch wrote is read before the wait.
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");

  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~(uintptr_t)1023);
  SmemBarriers* bars = reinterpret_cast<SmemBarriers*>(smem + kStages * kStageBytes);
  double* red = reinterpret_cast<double*>(smem);   // the ring is idle when the tail reduction runs

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const uint32_t rank = (CG == 2) ? cluster_ctarank() : 0u;
  const int cluster_id = blockIdx.x / CG;
  const bool leader = (rank == 0);

  const Sp2LayerArgs& a0 = args[0];       // everything but the planes / tensor maps is the same in both blocks
  const int n_tiles = a0.n_tiles;
  const int KB = a0.npad / kBK;            // ring stages per k sweep
  const int seg_kb = a0.seg_kb * (64 / kBK);   // ring stages per TMEM accumulation segment (divides KB)
  const int item_lo = a0.item_begin[cluster_id], item_hi = a0.item_begin[cluster_id + 1];
  const int nz_units = MODE == 1 ? 0 : a0.with_response * n_tiles;   // units [0, nz_units): first-order, then the Y^2 units

  if (warp == kWarpTma && lane == 0) {
    const int n_maps = MODE == 1 ? 4 : 2 + 2 * a0.with_response;
    for (int i = 0; i < n_maps; ++i) {
      asm volatile("prefetch.tensormap [%0];" ::"l"(&args[0].tm[i]) : "memory");
      if (PERSIST) asm volatile("prefetch.tensormap [%0];" ::"l"(&args[1].tm[i]) : "memory");
    }
  }
  if (warp == kWarpMma && lane == 0) {
    for (int s = 0; s < kStages; ++s) { mbar_init(smem_u32(&bars->full[s]), 1); mbar_init(smem_u32(&bars->empty[s]), 1); }
    for (int s = 0; s < 2; ++s) { mbar_init(smem_u32(&bars->tmem_full[s]), 1); mbar_init(smem_u32(&bars->tmem_empty[s]), kConsumerWarps * CG); }
    bars->stop = 0u; bars->prod_layers = 1u; bars->prod_final = 0u;
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp < kConsumerWarps && lane < 1 + SP2_NB) {
    Sp2Slot z; z.tr = 0.0; z.fro = 0.0; z.tracc = 0.0; z.mx = 0.f; z.pad = 0.f;
    bars->acc[warp][lane] = z;
  }
  if (warp == kWarpAlloc) tmem_alloc<CG>(smem_u32(&bars->tmem_base), TMEM_COLS);
  tc_fence_before();
  if constexpr (CG == 2) cluster_sync_all(); else __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *reinterpret_cast<volatile uint32_t*>(&bars->tmem_base);

  asm volatile("griddepcontrol.wait;" ::: "memory");    // previous layer complete, its writes visible
  const bool active = MODE == 1 || *reinterpret_cast<volatile const int*>(&a0.ctrl->done) == 0;   // uniform over the grid
  // persistent mode: the layer about to run fixes which buffer is read.  The controller has already counted it
  // (ctrl->n = its index + 1 while done == 0), so layer ctrl->n - 1 reads buffer (ctrl->n - 1) & 1.
  int par = PERSIST ? ((*reinterpret_cast<volatile const int*>(&a0.ctrl->n) + 1) & 1) : 0;
  // persistent mode: grid barriers passed before this launch (0 for the one launch of a solve: k_init clears the block)
  const unsigned int epoch0 = PERSIST ? ld_acquire_u32(&a0.ctrl->epoch) : 0u;

  if (!active) {
    // converged (or failed) before this launch: nothing to do but release the TMEM columns
  } else if (warp >= kConsumerWarps) {
    asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(kRegsProducer));
    if (warp == kWarpTma) {
      // =================================== TMA producer (one lane, every CTA) ==================
      if (elect_one()) {
        int stage = 0; uint32_t phase = 0;
        unsigned int layers_loaded = 0;
        bool lock_live = true;
        int cum = 0;                       // k-blocks issued inside the lockstep region of this launch
        uint32_t full_bar[kStages];
        for (int s = 0; s < kStages; ++s) {
          full_bar[s] = smem_u32(&bars->full[s]);
          if constexpr (CG == 2) asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(full_bar[s]) : "r"(full_bar[s]), "r"(0));
        }
        for (;;) {
          const Sp2LayerArgs& a = args[par];
          for (int iti = item_lo; iti < item_hi; ++iti) {
            const Sp2Item I = a.items[iti];
            const int u = I.unit;
            const bool wunit = u < nz_units;           // Y Z_b + Z_b Y unit of perturbation b = u / n_tiles
            const int zb = wunit ? u / n_tiles : 0;
            const int2 tij = a.tiles[wunit ? u - zb * n_tiles : u - nz_units];
            const int zpl = 2 + 2 * zb;                // planes of Z_b
            const int row_a = tij.x * TILE + (int)rank * kRows;
            const int row_b = tij.y * TILE + (int)rank * kRows;
            for (int g = I.seg0 * seg_kb; g < I.seg1 * seg_kb; ++g) {
              // Y^2: A = (Yh, Ym), B = (Yh, Ym).  W pass 0: A = (Yh, Ym), B = (Zh, Zm).  W pass 1: A = (Zh, Zm), B = (Yh, Ym).
              const int p = (g >= KB) ? 1 : 0;
              const int kb = g - p * KB;
              const int ma = (wunit && p == 1) ? zpl : 0;
              const int mb = (MODE == 1 || (wunit && p == 0)) ? zpl : 0;
              // Soft lockstep (launch-per-layer mode, large N): CTAs that run concurrently stream the same row / column
              // panels, and a panel byte is fetched from DRAM once only while they stay within an L2's worth of
              // k-blocks of one another.  Every kLockEvery k-blocks of its leading whole units a producer arrives on a
              // checkpoint counter and starts the next chunk only when lock_need of the grid's producers have arrived
              // there too (7/8 of them: one slow CTA does not stall the rest; the 3-stage ring hides short waits).
              // The wait is a hint, not a dependency: it gives up after lock_polls polls and this CTA then free-runs
              // for the rest of the launch, so a grid that is not fully resident (another stream's kernels on the same
              // SMs) loses the traffic saving, not its progress.
              if (!PERSIST && lock_live && cum < a.lock_kb && cum > 0 && (cum & (kLockEvery - 1)) == 0) {
                const volatile unsigned int* cnt = a.flags + a.n_flags + (cum / kLockEvery - 1);
                int polls = 0;
                while (*cnt < (unsigned)a.lock_need) {
                  if (++polls > a.lock_polls) { lock_live = false; break; }
                  __nanosleep(256);
                }
              }
              mbar_wait(smem_u32(&bars->empty[stage]), phase ^ 1u);
              const uint32_t dst = smem_u32(smem + stage * kStageBytes);
              if (CG == 1 || leader) mbar_expect_tx(smem_u32(&bars->full[stage]), (uint32_t)(CG * kStageBytes));
              tma_load_2d<CG>(dst + 0 * kPlaneTileBytes, &a.tm[ma + 0], full_bar[stage], kb * kBK, row_a);
              tma_load_2d<CG>(dst + 1 * kPlaneTileBytes, &a.tm[ma + 1], full_bar[stage], kb * kBK, row_a);
              tma_load_2d<CG>(dst + 2 * kPlaneTileBytes, &a.tm[mb + 0], full_bar[stage], kb * kBK, row_b);
              tma_load_2d<CG>(dst + 3 * kPlaneTileBytes, &a.tm[mb + 1], full_bar[stage], kb * kBK, row_b);
              if (++stage == kStages) { stage = 0; phase ^= 1u; }
              if (!PERSIST && cum < a.lock_kb) {
                ++cum;
                if ((cum & (kLockEvery - 1)) == 0) atomicAdd(a.flags + a.n_flags + (cum / kLockEvery - 1), 1u);
              }
            }
          }
          if (!PERSIST) break;
          // arrive half of the grid barrier: every CTA has stored its planes of the layer just loaded.  (When the
          // controller stops, no CTA arrives for the layer after: the consumers raise `stop` instead.  The ticket is
          // tested first, so the one speculative layer is ALWAYS started and the consumers always drain exactly one.)
          ++layers_loaded;
          bool more = false;
          for (long long spins = 0;; ++spins) {
            if (ld_acquire_u32(&a.ctrl->ticket) >= (epoch0 + layers_loaded) * gridDim.x) { more = true; break; }
            if (*reinterpret_cast<volatile const uint32_t*>(&bars->stop)) break;
            if (spins > kSpinLimit) __trap();
            __nanosleep(200);       // this warp shares a scheduler with two consumer warps (epilogue, controller)
          }
          if (!more) { *reinterpret_cast<volatile uint32_t*>(&bars->prod_final) = 1u; break; }
          fence_proxy_async_global();
          *reinterpret_cast<volatile uint32_t*>(&bars->prod_layers) = layers_loaded + 1u;
          par ^= 1;
        }
      }
    } else if (warp == kWarpMma) {
      // =================================== MMA issuer (one lane of the leader CTA) ==============
      if (leader && elect_one()) {
        int stage = 0; uint32_t phase = 0;
        unsigned int layers_issued = 0;
        int as = 0; uint32_t aphase = 0;
        for (;;) {
          for (int iti = item_lo; iti < item_hi; ++iti) {
            const Sp2Item I = a0.items[iti];
            for (int sg = I.seg0; sg < I.seg1; ++sg) {
              mbar_wait(smem_u32(&bars->tmem_empty[as]), aphase ^ 1u);
              tc_fence_after();
              const uint32_t acc = tmem_base + (uint32_t)(as * ACC_COLS);
              for (int it = 0; it < seg_kb; ++it) {
                mbar_wait(smem_u32(&bars->full[stage]), phase);
                tc_fence_after();
                const uint32_t sa = smem_u32(smem + stage * kStageBytes);
                const uint64_t dA0 = make_smem_desc(sa + 0 * kPlaneTileBytes);
                const uint64_t dA1 = make_smem_desc(sa + 1 * kPlaneTileBytes);
                const uint64_t dB0 = make_smem_desc(sa + 2 * kPlaneTileBytes);
                const uint64_t dB1 = make_smem_desc(sa + 3 * kPlaneTileBytes);
#pragma unroll
                for (int k = 0; k < kBK / 16; ++k) {
                  const uint64_t ko = (uint64_t)(k * 2);     // 16 elements * 2 B = 32 B -> >>4 = 2
                  // small cross terms first, the dominant hi*hi product last
                  // the two products with A.hi are adjacent: A.hi is read from shared memory once (collector buffer)
                  umma_f16<CG>(acc, dA1 + ko, dB0 + ko, IDESC, (it | k) ? 1u : 0u);
                  umma_f16<CG, 1>(acc, dA0 + ko, dB1 + ko, IDESC, 1u);
                  umma_f16<CG, 2>(acc, dA0 + ko, dB0 + ko, IDESC, 1u);
                }
                umma_commit<CG>(smem_u32(&bars->empty[stage]));   // smem slot free when these MMAs retire
                if (++stage == kStages) { stage = 0; phase ^= 1u; }
              }
              umma_commit<CG>(smem_u32(&bars->tmem_full[as]));     // segment accumulator complete
              if (++as == 2) { as = 0; aphase ^= 1u; }
            }
          }
          if (!PERSIST) break;
          ++layers_issued;                         // follow the producer: another layer, or the end
          bool more = false;
          for (long long spins = 0;; ++spins) {
            if (*reinterpret_cast<volatile const uint32_t*>(&bars->prod_layers) > layers_issued) { more = true; break; }
            if (*reinterpret_cast<volatile const uint32_t*>(&bars->prod_final)) break;
            if (spins > kSpinLimit) __trap();
            __nanosleep(100);
          }
          if (!more) break;
        }
      }
    }
  } else {
    // ===================================== consumer warps (8 per CTA) ===========================
    asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(kRegsConsumer));
    const int cw = warp;
    const int q = warp & 3;                       // TMEM lane quarter this warp may read
    const int hh = cw >> 2;                       // which half of the accumulator columns
    const double gemm_scale = MODE == 1 ? sp2_exp2i((a0.out_kind == 0 ? a0.ctrl->g_et : 0) - a0.ctrl->g_ea - a0.ctrl->g_eb) : 0.0;
    // optional power saving: round the lo plane to lo_bits significant bits (fewer toggling multiplier inputs)
    const int drop = 11 - a0.lo_bits;
    const uint32_t lo_mask = drop > 0 ? ~(((1u << drop) - 1u) * 0x00010001u) : 0xffffffffu;
    const uint32_t lo_round = drop > 0 ? (1u << (drop - 1)) * 0x00010001u : 0u;
    int as = 0; uint32_t aphase = 0;
    unsigned int epoch = epoch0;
    if constexpr (PERSIST) {                      // this CTA's working copy of the control block (history included)
      const uint32_t* src = reinterpret_cast<const uint32_t*>(a0.ctrl);
      uint32_t* dst = reinterpret_cast<uint32_t*>(bars->ctrl_copy);
      for (int i = threadIdx.x; i < (int)(sizeof(Sp2Ctrl) / 4); i += kConsumerWarps * 32) dst[i] = __ldcg(src + i);
      named_bar_sync(1, kConsumerWarps * 32);
    }
    for (;;) {
    const Sp2LayerArgs& a = args[par];
    // persistent mode: the coefficients come from this CTA's copy, rewritten by its thread 0 between layers
    const volatile Sp2Coef* cz = PERSIST ? &reinterpret_cast<const volatile Sp2Ctrl*>(bars->ctrl_copy)->coef : &a.ctrl->coef;
    const float cf_a1y_hi = cz->a1y_hi, cf_a1y_lo = cz->a1y_lo, cf_a2y = cz->a2y;
    const float cf_dsh_hi = cz->dsh_hi, cf_dsh_lo = cz->dsh_lo;
    for (int iti = item_lo; iti < item_hi; ++iti) {
      const Sp2Item I = a.items[iti];
      const int u = I.unit;
      const bool wunit = u < nz_units;
      const int zb = wunit ? u / n_tiles : 0;
      const int2 tij = a.tiles[wunit ? u - zb * n_tiles : u - nz_units];
      float sums[WCOLS];
      const int pl = wunit ? 2 + 2 * zb : 0;
      const int gi = tij.x * TILE + (int)rank * kRows + q * 32 + lane;   // global row of this thread
      const int j0 = tij.y * TILE + hh * WCOLS;
      EpiOld old;
#pragma unroll 1
      for (int sg = I.seg0, ho = 0; sg < I.seg1; ++sg, ++ho) {
        // the old tile's first chunk is fetched under the last segment's MMAs
        if (MODE == 0 && sg + 1 == I.seg1 && I.kind != 1) epilogue_prefetch(old, gi, j0, (size_t)a.npad, a.in[pl], a.in[pl + 1]);
        mbar_wait(smem_u32(&bars->tmem_full[as]), aphase);
        tc_fence_after();
        const uint32_t tcol = tmem_base + ((uint32_t)(q * 32) << 16) + (uint32_t)(as * ACC_COLS + hh * WCOLS);
        if (ho == 0) {
#pragma unroll
          for (int ch = 0; ch < NCH; ++ch) {
            uint32_t v[32];
            tmem_ld32(tcol + ch * 32, v);
#pragma unroll
            for (int i = 0; i < 32; ++i) sums[ch * 32 + i] = __uint_as_float(v[i]);
          }
        } else {
#pragma unroll
          for (int ch = 0; ch < NCH; ++ch) {
            uint32_t v[32];
            tmem_ld32(tcol + ch * 32, v);
#pragma unroll
            for (int i = 0; i < 32; ++i) sums[ch * 32 + i] += __uint_as_float(v[i]);
          }
        }
        tc_fence_before();
        __syncwarp();
        if (lane == 0) {
          if constexpr (CG == 2) mbar_arrive_cluster(smem_u32(&bars->tmem_empty[as]), 0);
          else mbar_arrive(smem_u32(&bars->tmem_empty[as]));
        }
        if (++as == 2) { as = 0; aphase ^= 1u; }
      }
      // ---- split-k units of the last wave: hand the partial sums over / collect them
      constexpr size_t kWarpFloats = (size_t)WCOLS * 32;
      if (I.kind == 1) {
        float* dst = a.scratch + (((size_t)I.slot * CG + rank) * kConsumerWarps + cw) * kWarpFloats + lane;
#pragma unroll
        for (int c = 0; c < WCOLS; ++c) dst[c * 32] = sums[c];       // lanes contiguous: 128 B per store
        __syncwarp();
        // (split-k flags: two sets in persistent mode, used by alternate layers; block 0 re-arms the set just consumed)
        if (lane == 0) { __threadfence(); atomicAdd(a.flags + (PERSIST ? (epoch & 1u) * (unsigned int)a.n_flags : 0u) + I.flag_id, 1u); }
        continue;
      }
      if (I.kind == 2) {
        if (lane == 0) {
          const unsigned int target = (unsigned int)(I.nparts * kConsumerWarps * CG);
          long long spins = 0;
          const volatile unsigned int* fl = a.flags + (PERSIST ? (epoch & 1u) * (unsigned int)a.n_flags : 0u) + I.flag_id;
          while (*fl < target)
            if (++spins > kSpinLimit) __trap();
          __threadfence();
        }
        __syncwarp();
        for (int pp = 0; pp < I.nparts; ++pp) {
          const float* src = a.scratch + (((size_t)(I.slot + pp) * CG + rank) * kConsumerWarps + cw) * kWarpFloats + lane;
#pragma unroll
          for (int c = 0; c < WCOLS; ++c) sums[c] += __ldcg(src + c * 32);
        }
      }
      if constexpr (MODE == 1) {                  // plain product: scale, (split,) store; no statistics
        gemm_epilogue<WCOLS>(sums, gi, j0, a, gemm_scale);
        continue;
      }
      // ---- fused epilogue from the register sums
      const float a1hi = wunit ? cz->a1z_hi[zb] : cf_a1y_hi, a1lo = wunit ? cz->a1z_lo[zb] : cf_a1y_lo;
      const float a2 = wunit ? cz->a2z[zb] : cf_a2y;
      const bool shift_row = !wunit && gi < a.n;        // zero padding stays zero
      const float dsh_hi = shift_row ? cf_dsh_hi : 0.f, dsh_lo = shift_row ? cf_dsh_lo : 0.f;
      EpiPartials P; P.tr = 0.0; P.fro = 0.0; P.tracc = 0.0; P.mx = 0.f;
      epilogue_row<NCH>(sums, old, gi, j0, (size_t)a.npad, a.in[pl], a.in[pl + 1], a.out[pl], a.out[pl + 1],
                        a1hi, a1lo, a2, dsh_hi, dsh_lo, lo_round, lo_mask, bars->diag_t[q], P);
      // warp partial -> slot (fixed shuffle tree: deterministic)
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) {
        P.tr += __shfl_xor_sync(0xffffffffu, P.tr, o);
        P.fro += __shfl_xor_sync(0xffffffffu, P.fro, o);
        P.tracc += __shfl_xor_sync(0xffffffffu, P.tracc, o);
        const float qv = __shfl_xor_sync(0xffffffffu, P.mx, o);
        P.mx = (qv > P.mx || qv != qv) ? qv : P.mx;
      }
      if (lane == 0) {                           // fixed item order per warp: deterministic
        Sp2Slot& s = bars->acc[cw][wunit ? 1 + zb : 0];
        s.tr += P.tr; s.fro += P.fro;
        if (!wunit) s.tracc += P.tracc;
        s.mx = (P.mx > s.mx || P.mx != P.mx) ? P.mx : s.mx;   // NaN-propagating max
      }
    }
    if constexpr (!PERSIST) {
      break;
    } else {
      // ================================ end of a layer: grid-wide barrier ======================
      constexpr int NT = kConsumerWarps * 32;
      const int nb = a.with_response;
      const int nblk = (int)gridDim.x;
      fence_proxy_async_global();                  // this thread's plane stores -> visible to the next layer's TMA loads
      __threadfence();
      named_bar_sync(1, NT);
      // one slot per CTA and class: [z_0 .. z_{nb-1}][y], gridDim.x each; two sets, used by alternate layers (a fast
      // CTA may write the next layer's slots while a slow one still reads this layer's)
      Sp2Slot* const lslots = a.slots + (size_t)(epoch & 1u) * (size_t)(1 + nb) * nblk;
      if ((int)threadIdx.x < 1 + nb) {
        const int cls = threadIdx.x;
        Sp2Slot t = bars->acc[0][cls];
        for (int w = 1; w < kConsumerWarps; ++w) {
          const Sp2Slot& o = bars->acc[w][cls];
          t.tr += o.tr; t.fro += o.fro; t.tracc += o.tracc;
          t.mx = (o.mx > t.mx || o.mx != o.mx) ? o.mx : t.mx;
        }
        lslots[(size_t)(cls == 0 ? nb : cls - 1) * nblk + blockIdx.x] = t;
        Sp2Slot z; z.tr = 0.0; z.fro = 0.0; z.tracc = 0.0; z.mx = 0.f; z.pad = 0.f;
        for (int w = 0; w < kConsumerWarps; ++w) bars->acc[w][cls] = z;
        __threadfence();
      }
      named_bar_sync(1, NT);
      ++epoch;
      if (threadIdx.x == 0) {                      // the ticket only grows: epoch * nblk tickets end layer `epoch`
        atomicAdd(&a.ctrl->ticket, 1u);
        long long spins = 0;
        while ((int)(ld_acquire_u32(&a.ctrl->ticket) - epoch * (unsigned int)nblk) < 0)
          if (++spins > kSpinLimit) __trap();
        __threadfence();
      }
      named_bar_sync(1, NT);
      if (blockIdx.x == 0) {                       // every split unit of the layer was consumed: re-arm its flag set
        unsigned int* const used_flags = a.flags + ((epoch - 1u) & 1u) * (unsigned int)a.n_flags;
        for (int i = threadIdx.x; i < a.n_flags; i += NT) used_flags[i] = 0u;
        __threadfence();                           // ordered before this CTA's next ticket, which gates the set's next use
      }
      persist_control(a, bars, a.slots + (size_t)((epoch - 1u) & 1u) * (size_t)(1 + nb) * nblk, nb, nblk);
      Sp2Ctrl* const lctrl = reinterpret_cast<Sp2Ctrl*>(bars->ctrl_copy);
      const int done = *reinterpret_cast<volatile const int*>(&lctrl->done);
      if (done) {
        if (blockIdx.x == 0) {                     // the final control block -> global memory (read by the finalise kernels)
          if (threadIdx.x == 0) { lctrl->epoch = epoch; lctrl->ticket = epoch * (unsigned int)nblk; }
          named_bar_sync(1, NT);
          const uint32_t* src = reinterpret_cast<const uint32_t*>(lctrl);
          uint32_t* dst = reinterpret_cast<uint32_t*>(a.ctrl);
          for (int i = threadIdx.x; i < (int)(SP2_CTRL_HEAD_BYTES / 4); i += NT) dst[i] = src[i];
          __threadfence();
        }
        // the producer and the tensor core have started one more layer (see above): drain it, no epilogue
        if (threadIdx.x == 0) *reinterpret_cast<volatile uint32_t*>(&bars->stop) = 1u;
        for (int iti = item_lo; iti < item_hi; ++iti) {
          const Sp2Item I = a.items[iti];
          for (int sg = I.seg0; sg < I.seg1; ++sg) {
            mbar_wait(smem_u32(&bars->tmem_full[as]), aphase);
            tc_fence_after();
            tc_fence_before();
            __syncwarp();
            if (lane == 0) {
              if constexpr (CG == 2) mbar_arrive_cluster(smem_u32(&bars->tmem_empty[as]), 0);
              else mbar_arrive(smem_u32(&bars->tmem_empty[as]));
            }
            if (++as == 2) { as = 0; aphase ^= 1u; }
          }
        }
        break;
      }
      par ^= 1;
    }
    }
  }

  // ===================================== teardown ==============================================
  tc_fence_before();
  if constexpr (CG == 2) cluster_sync_all(); else __syncthreads();
  if (warp == kWarpAlloc) tmem_dealloc<CG>(tmem_base, TMEM_COLS);
  if (!active || PERSIST) return;
  const Sp2LayerArgs& a = a0;
  if constexpr (MODE == 1) {                     // last CTA re-arms the split-k flags; no controller
    __syncthreads();
    if (threadIdx.x == 0) {
      __threadfence();
      bars->is_last = (atomicAdd(&a.ctrl->ticket, 1u) == gridDim.x - 1) ? 1u : 0u;
    }
    __syncthreads();
    if (bars->is_last) {
      for (int i = threadIdx.x; i < a.n_flags + a.lock_kb / kLockEvery; i += blockDim.x) a.flags[i] = 0u;
      if (threadIdx.x == 0) a.ctrl->ticket = 0u;
    }
    return;
  }

  // one slot per CTA and class: [class z_0: gridDim.x slots] ... [class z_{nb-1}][class y]
  if ((int)threadIdx.x < 1 + a.with_response) {
    const int cls = threadIdx.x;               // 0: y, 1 + b: z_b
    Sp2Slot t = bars->acc[0][cls];
    for (int w = 1; w < kConsumerWarps; ++w) {
      const Sp2Slot& o = bars->acc[w][cls];
      t.tr += o.tr; t.fro += o.fro; t.tracc += o.tracc;
      t.mx = (o.mx > t.mx || o.mx != o.mx) ? o.mx : t.mx;
    }
    a.slots[(size_t)(cls == 0 ? a.with_response : cls - 1) * gridDim.x + blockIdx.x] = t;
  }
  layer_tail(a.ctrl, a.slots, gridDim.x, gridDim.x, a.with_response, gridDim.x, &bars->is_last, red, a.flags,
             a.n_flags + a.lock_kb / kLockEvery);
}


template <int CG, int MODE>
__global__ void __launch_bounds__(kThreads, 1) k_layer_tc(const __grid_constant__ Sp2LayerArgs a) {
  layer_body<CG, MODE, false>(&a);
}

// args: the two argument blocks (TMA descriptors included) in GLOBAL memory, written by the host before the launch
template <int CG>
__global__ void __launch_bounds__(kThreads, 1) k_layers_persist(const Sp2LayerArgs* __restrict__ args) {
  layer_body<CG, 0, true>(args);
}

// ----------------------------------------------------------------------------------------------
// SIMT debug engine (tests only): same planes, same unit semantics, same epilogue element function,
// plain FP32 FMA mainloop.  16x16 output elements per block, blockIdx.y = product class.
__global__ void __launch_bounds__(256) k_layer_simt(Sp2LayerArgs a) {
  if (a.ctrl->done) return;
  __shared__ double red[4 * 256];
  __shared__ uint32_t is_last;
  __shared__ double rs[3][8];
  __shared__ float rm[8];
  const int nb = a.npad / 16;
  const int n_blk_tri = nb * (nb + 1) / 2;
  const int cls = blockIdx.y;                  // 0: Y^2, 1 + b: Y Z_b + Z_b Y
  int bi = 0, rem = blockIdx.x;
  while (rem >= nb - bi) { rem -= nb - bi; ++bi; }
  const int bj = bi + rem;
  const int r = threadIdx.x >> 4, cidx = threadIdx.x & 15;
  const int gi = bi * 16 + r, gj = bj * 16 + cidx;
  const size_t npad = (size_t)a.npad;
  const __half* Yh = a.in[0]; const __half* Ym = a.in[1];
  const __half* Zh = a.in[2 * cls]; const __half* Zm = a.in[2 * cls + 1];
  float acc = 0.f;
  if (cls == 0) {
    for (int k = 0; k < a.npad; ++k) {
      const float hi_ = __half2float(Yh[gi * npad + k]), mi = __half2float(Ym[gi * npad + k]);
      const float hj = __half2float(Yh[gj * npad + k]), mj = __half2float(Ym[gj * npad + k]);
      acc = fmaf(hi_, hj, acc); acc = fmaf(hi_, mj, acc); acc = fmaf(mi, hj, acc);
    }
  } else {
    for (int k = 0; k < a.npad; ++k) {
      const float hi_ = __half2float(Yh[gi * npad + k]), mi = __half2float(Ym[gi * npad + k]);
      const float hj = __half2float(Yh[gj * npad + k]), mj = __half2float(Ym[gj * npad + k]);
      const float pi_ = __half2float(Zh[gi * npad + k]), qi = __half2float(Zm[gi * npad + k]);
      const float pj = __half2float(Zh[gj * npad + k]), qj = __half2float(Zm[gj * npad + k]);
      acc = fmaf(hi_, pj, acc); acc = fmaf(hi_, qj, acc); acc = fmaf(mi, pj, acc);
      acc = fmaf(pi_, hj, acc); acc = fmaf(pi_, mj, acc); acc = fmaf(qi, hj, acc);
    }
  }
  const Sp2Coef& cf = a.ctrl->coef;
  const int pl = 2 * cls;
  const int zb = cls ? cls - 1 : 0;
  const float a1hi = cls ? cf.a1z_hi[zb] : cf.a1y_hi, a1lo = cls ? cf.a1z_lo[zb] : cf.a1y_lo, a2 = cls ? cf.a2z[zb] : cf.a2y;
  double tr = 0.0, fro = 0.0, tracc = 0.0;
  float mx = 0.f;
  if (gj >= gi) {
    const float old = __half2float(a.in[pl][gi * npad + gj]) + __half2float(a.in[pl + 1][gi * npad + gj]);
    __half nh, nm;
    const bool dg = (gj == gi) && cls == 0 && gi < a.n;
    const float s = sp2_epilogue_elem(old, acc, a1hi, a1lo, a2, dg ? cf.dsh_hi : 0.f, dg ? cf.dsh_lo : 0.f, nh, nm);
    a.out[pl][gi * npad + gj] = nh; a.out[pl + 1][gi * npad + gj] = nm;
    if (gj > gi) { a.out[pl][gj * npad + gi] = nh; a.out[pl + 1][gj * npad + gi] = nm; }
    fro = (gj > gi ? 2.0 : 1.0) * (double)s * (double)s;
    if (gj == gi) { tr = (double)s; if (cls == 0) tracc = (double)acc; }
    mx = (s != s) ? s : fabsf(s);
  }
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    tr += __shfl_xor_sync(0xffffffffu, tr, o);
    fro += __shfl_xor_sync(0xffffffffu, fro, o);
    tracc += __shfl_xor_sync(0xffffffffu, tracc, o);
    const float qv = __shfl_xor_sync(0xffffffffu, mx, o);
    mx = (qv > mx || qv != qv) ? qv : mx;
  }
  if (lane == 0) { rs[0][warp] = tr; rs[1][warp] = fro; rs[2][warp] = tracc; rm[warp] = mx; }
  __syncthreads();
  if (threadIdx.x == 0) {
    Sp2Slot s; s.tr = 0; s.fro = 0; s.tracc = 0; s.mx = 0.f; s.pad = 0.f;
    for (int w = 0; w < 8; ++w) { s.tr += rs[0][w]; s.fro += rs[1][w]; s.tracc += rs[2][w]; s.mx = (rm[w] > s.mx || rm[w] != rm[w]) ? rm[w] : s.mx; }
    // layout [z slots of perturbation 0] ... [z slots of perturbation nb - 1][y slots]
    a.slots[(size_t)(cls ? cls - 1 : a.with_response) * n_blk_tri + blockIdx.x] = s;
  }
  layer_tail(a.ctrl, a.slots, n_blk_tri, n_blk_tri, a.with_response, gridDim.x * gridDim.y, &is_last, red);
}

}  // namespace

// ----------------------------------------------------------------------------------------------
int sp2_layer_box_k() { return kBK; }

size_t sp2_layer_smem_bytes() { return (size_t)kStages * kStageBytes + sizeof(SmemBarriers) + 1024; }

// Partial-sum slots one layer launch writes: the tcgen05 engine writes ONE slot per CTA and product class at
// class * gridDim.x + blockIdx.x (k_layer_tc, end of the kernel), so it needs (1 + nb) * grid_ctas; the SIMT
// scaffold writes one per 16x16 block and class.
int sp2_layer_slots(int npad, int grid_ctas, int with_response, int engine) {
  if (engine == SP2_ENGINE_SIMT_DEBUG) {
    const int nb = npad / 16;
    return nb * (nb + 1) / 2 * (1 + with_response);
  }
  return 2 * grid_ctas * (1 + with_response);   // two sets: the persistent mode alternates them between layers
}

cudaError_t sp2_layer_configure() {
  const int smem = (int)sp2_layer_smem_bytes();
  cudaError_t e = cudaFuncSetAttribute(k_layer_tc<1, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
  if (e == cudaSuccess) e = cudaFuncSetAttribute(k_layer_tc<2, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
  if (e == cudaSuccess) e = cudaFuncSetAttribute(k_layer_tc<1, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
  if (e == cudaSuccess) e = cudaFuncSetAttribute(k_layer_tc<2, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
  if (e == cudaSuccess) e = cudaFuncSetAttribute(k_layers_persist<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
  if (e == cudaSuccess) e = cudaFuncSetAttribute(k_layers_persist<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
  return e;
}

// CTAs (cta_group 1) or CTA pairs (cta_group 2) of the layer kernel the current device can keep resident at once
// (static resources only: registers, 200 KB of shared memory, cluster placement inside the GPCs).
cudaError_t sp2_layer_max_coresident(int cta_group, int num_sms, int* out) {
  *out = 0;
  if (cta_group == 2) {
    cudaLaunchConfig_t cfg = {};
    cfg.blockDim = dim3(kThreads);
    cfg.gridDim = dim3(2 * (num_sms / 2));
    cfg.dynamicSmemBytes = sp2_layer_smem_bytes();
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = 2; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr; cfg.numAttrs = 1;
    return cudaOccupancyMaxActiveClusters(out, k_layer_tc<2, 0>, &cfg);
  }
  int per_sm = 0;
  cudaError_t e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_layer_tc<1, 0>, kThreads, sp2_layer_smem_bytes());
  *out = per_sm * num_sms;
  return e;
}

size_t sp2_layer_scratch_slot_bytes(int cta_group) {
  return (size_t)cta_group * kConsumerWarps * (128 * cta_group / 2) * 32 * sizeof(float);
}

cudaError_t sp2_launch_layer(const Sp2LayerArgs& args, int engine, int cta_group, cudaStream_t s) {
  if (engine == SP2_ENGINE_SIMT_DEBUG) {
    const int nb = args.npad / 16;
    dim3 grid(nb * (nb + 1) / 2, 1 + args.with_response);
    k_layer_simt<<<grid, 256, 0, s>>>(args);
    return cudaGetLastError();
  }
  cudaLaunchConfig_t cfg = {};
  cfg.blockDim = dim3(kThreads);
  cfg.dynamicSmemBytes = sp2_layer_smem_bytes();
  cfg.stream = s;
  cudaLaunchAttribute attr[2];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;    // PDL: see the top of k_layer_tc
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr; cfg.numAttrs = 1;
  if (cta_group == 2) {
    cfg.gridDim = dim3(2 * args.n_clusters);
    attr[1].id = cudaLaunchAttributeClusterDimension;
    attr[1].val.clusterDim.x = 2; attr[1].val.clusterDim.y = 1; attr[1].val.clusterDim.z = 1;
    cfg.numAttrs = 2;
    return args.gemm_mode ? cudaLaunchKernelEx(&cfg, k_layer_tc<2, 1>, args) : cudaLaunchKernelEx(&cfg, k_layer_tc<2, 0>, args);
  }
  cfg.gridDim = dim3(args.n_clusters);
  return args.gemm_mode ? cudaLaunchKernelEx(&cfg, k_layer_tc<1, 1>, args) : cudaLaunchKernelEx(&cfg, k_layer_tc<1, 0>, args);
}

// The whole layer stack in ONE launch (persistent multi-layer mode): d_args = two argument blocks in DEVICE memory
// (d_args[0] reads buffer 0 and writes buffer 1, d_args[1] the reverse); `grid_clusters` CTA(-pair)s (those with
// work), all of which must be co-resident.
cudaError_t sp2_launch_layers_persistent(const Sp2LayerArgs* d_args, int cta_group, int grid_clusters, cudaStream_t s) {
  cudaLaunchConfig_t cfg = {};
  cfg.blockDim = dim3(kThreads);
  cfg.dynamicSmemBytes = sp2_layer_smem_bytes();
  cfg.stream = s;
  cudaLaunchAttribute attr[1];
  cfg.attrs = attr; cfg.numAttrs = 0;
  if (cta_group == 2) {
    cfg.gridDim = dim3(2 * grid_clusters);
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = 2; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, k_layers_persist<2>, d_args);
  }
  cfg.gridDim = dim3(grid_clusters);
  return cudaLaunchKernelEx(&cfg, k_layers_persist<1>, d_args);
}
