// sp2_small.cu -- a SMALL problem (N <= 128) solved by ONE CTA with the iterate resident in shared memory
// ("N <= 256: whole problem in one CTA's smem, all layers in one launch").
//
// At this size a layer is ~1 us of tensor work; what the multi-CTA kernels pay per layer -- global-memory round
// trips for the planes, a grid-wide barrier, the cross-CTA reduction -- is ten times that, and the seven short
// kernels around the stack (bounds, set-up, rescale, controller, finalise) cost as much as the stack itself.  Here
// nothing leaves the SM between layers, and k_small_solve runs the WHOLE solve in one launch:
//   a1/a2    Gershgorin discs, tr H, non-finite check, X_0 = (eps_max I - H)/Delta as c_0 I + Y_0, Z_0 = -H1/Delta,
//            FP16 hi/lo split straight into shared memory
//   planes   Yh, Ym (and Zh_b, Zm_b for up to two perturbations) live in shared memory in the K-major SWIZZLE_128B
//            layout tcgen05.mma reads (two 128-row x 64-k boxes per plane) and are updated IN PLACE: a layer's MMAs
//            have all retired before its epilogue writes, and only the thread that owns an upper-triangle element
//            ever reads its old value;
//   a3       tcgen05.mma 128x128x16 kind::f16, FP32 accumulators in TMEM (128 columns for Y^2, 128 more per
//            perturbation for Y Z_b + Z_b Y): the same three plane products per k-step as the large kernel
//            (Eq. 20-22: X = X^(0) + X^(1), the lo*lo term dropped); K = 128 is one accumulation
//            segment (24 MMAs, fewer than the 96 of the large kernel's segments: DESIGN.md "truncation bias");
//   a4       tcgen05.ld -> registers -> update, hi/lo split, element (i,j) and its mirror (j,i) written to shared
//            memory (bit-symmetric planes), partial sums; 8 warps, up to two 32 x 32 blocks of the upper triangle each
//            (16 warps with one block each measured slower: 128 instead of 255 registers per thread);
//   a5       block-wide reduction of the partial sums, then ONE thread runs the SAME controller as every other path
//            (sp2_controller: trace rule, stop test, shift, exponents) on a shared-memory copy of the control block,
//            while another warp already issues the next layer's MMAs (they need the planes, not the decision);
//   a6       D = c I + Y, D1_b = Z_b in the caller's dtype, tr D, tr(DH), tr D1_b, result struct.
// k_small_stack is the layer stack alone (a3-a5), used when the prologue must run as separate kernels (Lanczos bounds).
// Both leave the final planes and the control block in the workspace, where the debug hooks and the float64
// refinement expect them.
#include <cuda.h>
#include <cstring>
#include <mutex>
#include "sp2_internal.cuh"
#include "sp2_layer.h"
#include "sp2_ptx.cuh"

namespace {
using namespace sp2ptx;

constexpr int kNs = 128;                        // padded dimension of the small path (one UMMA tile)
constexpr int kBoxK = 64;                       // k extent of a TMA box (= sp2_layer_box_k())
constexpr int kBoxBytesS = kNs * kBoxK * 2;     // 16 KB: 128 rows x 128 bytes
constexpr int kPlaneBytesS = 2 * kBoxBytesS;    // 32 KB: k-blocks 0 and 1
constexpr int kThreadsS = 256;                  // 8 warps: TMEM lane quarter = warp & 3, column half = warp >> 2 (two 32-column chunks)
constexpr int kWarpsS = kThreadsS / 32;
constexpr int kMaxNbS = 2;                      // perturbations: planes (2 + 2 nb) x 32 KB <= 192 KB, TMEM (1 + nb) x 128 <= 512
constexpr int kWarpIssue = 3;                   // warp (quarter 3, columns 0..63) lies below the diagonal: no epilogue work,
constexpr int kWarpAllocS = 3;                  //   so MMA issue and TMEM allocation live there

struct SmallShared {
  uint64_t bar_load, bar_mma;
  uint32_t tmem_base, pad;
  double red[1 + kMaxNbS][3][kWarpsS];          // per class and warp: tr, fro, tracc
  float redm[1 + kMaxNbS][kWarpsS];
  double red2[8][kWarpsS];                      // prologue / finalise reductions
  alignas(8) uint8_t ctrl[sizeof(Sp2Ctrl)];
};

// byte offset of element (row, k) inside a plane: box k / 64, 128-byte rows, 16-byte chunks XORed with row & 7
// (the SWIZZLE_128B pattern of the TMA box; box bases are 1024-byte aligned)
__device__ __forceinline__ uint32_t sw_off(int row, int k) {
  const int kk = k & 63;
  return (uint32_t)((k >> 6) * kBoxBytesS + row * 128 + ((((kk >> 3) ^ (row & 7))) << 4) + ((kk & 7) << 1));
}

__device__ __forceinline__ float2 h2f2(uint32_t w) { return __half22float2(*reinterpret_cast<const __half2*>(&w)); }
__device__ __forceinline__ uint32_t f2h2(float a, float b) {
  const __half2 h = __floats2half2_rn(a, b);
  return *reinterpret_cast<const uint32_t*>(&h);
}
__device__ __forceinline__ uint32_t u4w(const uint4& v, int i) { return i == 0 ? v.x : (i == 1 ? v.y : (i == 2 ? v.z : v.w)); }

// One product class of one layer for this thread's row gi and ONE 32-column chunk gj0 .. gj0 + 31 on or above the
// diagonal: new values from the accumulators and the old planes, written in place (element and mirror), partial sums.
//   Ph, Pm: the class's hi / lo planes in shared memory.  diag: the chunk is this warp's 32 x 32 diagonal block.
__device__ __forceinline__ void small_epilogue(uint32_t tcol, uint8_t* Ph, uint8_t* Pm, int gi, int gj0, int lane, bool diag,
                                               float a1hi, float a1lo, float a2, float dsh_hi, float dsh_lo,
                                               uint32_t lo_round, uint32_t lo_mask,
                                               double& tr, double& fro, double& tracc, float& mxo) {
  float fsum = 0.f, mx = mxo, dval = 0.f, dacc = 0.f;
  uint32_t v[32];
  tmem_ld32(tcol, v);
  uint32_t nh[16], nm[16];
#pragma unroll
  for (int w = 0; w < 4; ++w) {
    const uint4 oh = *reinterpret_cast<const uint4*>(Ph + sw_off(gi, gj0 + 8 * w));
    const uint4 om = *reinterpret_cast<const uint4*>(Pm + sw_off(gi, gj0 + 8 * w));
#pragma unroll
    for (int pr = 0; pr < 4; ++pr) {
      const int ci = 8 * w + 2 * pr;
      const float2 fh = h2f2(u4w(oh, pr)), fm = h2f2(u4w(om, pr));
      const float acc0 = __uint_as_float(v[ci]), acc1 = __uint_as_float(v[ci + 1]);
      float y0 = fmaf(a1hi, fh.x + fm.x, fmaf(a1lo, fh.x + fm.x, a2 * acc0));
      float y1 = fmaf(a1hi, fh.y + fm.y, fmaf(a1lo, fh.y + fm.y, a2 * acc1));
      if (diag && ci == lane) { y0 = (y0 + dsh_lo) + dsh_hi; dacc = acc0; }
      if (diag && ci + 1 == lane) { y1 = (y1 + dsh_lo) + dsh_hi; dacc = acc1; }
      const uint32_t h = f2h2(y0, y1);
      const float2 hb = h2f2(h);
      const uint32_t m = (f2h2(y0 - hb.x, y1 - hb.y) + lo_round) & lo_mask;
      nh[4 * w + pr] = h; nm[4 * w + pr] = m;
      const float2 mb = h2f2(m);
      const float s0 = hb.x + mb.x, s1 = hb.y + mb.y;    // the values the next layer will see
      // weights: above the diagonal twice (the mirror image), on it once, below it not at all (diagonal block only)
      const float w0 = !diag ? 2.f : (ci > lane ? 2.f : (ci == lane ? 1.f : 0.f));
      const float w1 = !diag ? 2.f : (ci + 1 > lane ? 2.f : (ci + 1 == lane ? 1.f : 0.f));
      fsum = fmaf(w0 * s0, s0, fsum);
      fsum = fmaf(w1 * s1, s1, fsum);
      if (w0 != 0.f) mx = fmaxf(mx, fabsf(s0));
      if (w1 != 0.f) mx = fmaxf(mx, fabsf(s1));
      if (diag && ci == lane) dval = s0;
      if (diag && ci + 1 == lane) dval = s1;
    }
    // this row, 8 columns: one 16-byte store per plane (the part left of the diagonal is overwritten below)
    *reinterpret_cast<uint4*>(Ph + sw_off(gi, gj0 + 8 * w)) = make_uint4(nh[4 * w], nh[4 * w + 1], nh[4 * w + 2], nh[4 * w + 3]);
    *reinterpret_cast<uint4*>(Pm + sw_off(gi, gj0 + 8 * w)) = make_uint4(nm[4 * w], nm[4 * w + 1], nm[4 * w + 2], nm[4 * w + 3]);
  }
  if (diag) __syncwarp();                         // rows of the block first, then the mirror images over their left parts
  // mirror image (gj, gi): lanes = consecutive k of one row -> 64 contiguous bytes per store
#pragma unroll
  for (int c = 0; c < 32; ++c) {
    if (!diag || c > lane) {
      const uint32_t hw = nh[c >> 1], mw = nm[c >> 1];
      const unsigned short hv = (unsigned short)((c & 1) ? (hw >> 16) : (hw & 0xffffu));
      const unsigned short mv = (unsigned short)((c & 1) ? (mw >> 16) : (mw & 0xffffu));
      const uint32_t o = sw_off(gj0 + c, gi);
      *reinterpret_cast<unsigned short*>(Ph + o) = hv;
      *reinterpret_cast<unsigned short*>(Pm + o) = mv;
    }
  }
  mxo = mx;
  fro += (double)fsum;
  tr += (double)dval;
  tracc += (double)dacc;
}

// ---- block-wide reductions over the 16 warps: fixed shuffle tree, then the warp partials in index order (deterministic).
// Every thread returns the result.  `slot`: which row of sh->red2 to use (callers use a different row per call between
// two __syncthreads of their own).
__device__ __forceinline__ double block_sum(double v, SmallShared* sh, int slot) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  if ((threadIdx.x & 31) == 0) sh->red2[slot][threadIdx.x >> 5] = v;
  __syncthreads();
  double t = 0.0;
  for (int w = 0; w < kWarpsS; ++w) t += sh->red2[slot][w];
  return t;
}
__device__ __forceinline__ double block_max(double v, SmallShared* sh, int slot) {   // NaN-propagating
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) { const double q = __shfl_xor_sync(0xffffffffu, v, o); v = (q > v || q != q) ? q : v; }
  if ((threadIdx.x & 31) == 0) sh->red2[slot][threadIdx.x >> 5] = v;
  __syncthreads();
  double t = sh->red2[slot][0];
  for (int w = 1; w < kWarpsS; ++w) { const double q = sh->red2[slot][w]; t = (q > t || q != q) ? q : t; }
  return t;
}
__device__ __forceinline__ double block_min(double v, SmallShared* sh, int slot) { return -block_max(-v, sh, slot); }

// ---- the layer stack (a3-a5) on the planes in shared memory; ctrl (shared memory) holds the controller's decision
// for the first layer on entry.  All threads.
__device__ __forceinline__ void small_run_stack(uint8_t* smem, SmallShared* sh, Sp2Ctrl* ctrl, int nb, int n, int lo_bits,
                                                uint32_t tmem_base) {
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  constexpr uint32_t IDESC = make_idesc(kNs, kNs);
  const int q = warp & 3, hh = warp >> 2;
  const int gi = q * 32 + lane;                    // this thread's row = its TMEM lane
  const bool has_work = 2 * hh + 1 >= q;           // blocks below the diagonal are the mirror images of those above
  const int drop = 11 - lo_bits;
  const uint32_t lo_mask = drop > 0 ? ~(((1u << drop) - 1u) * 0x00010001u) : 0xffffffffu;
  const uint32_t lo_round = drop > 0 ? (1u << (drop - 1)) * 0x00010001u : 0u;
  uint32_t mma_phase = 0;

  // products of one layer: Y^2 -> columns [0, 128); Y Z_b + Z_b Y -> columns [128 (1 + b), +128).  One elected thread.
  auto issue_products = [&]() {
    tc_fence_after();
    const uint32_t sY = smem_u32(smem);
    for (int cls = 0; cls <= nb; ++cls) {
      const uint32_t sZ = smem_u32(smem + (size_t)(2 * cls) * kPlaneBytesS);
      const uint32_t acc = tmem_base + (uint32_t)(cls * kNs);
      const int passes = cls == 0 ? 1 : 2;        // W: (Y, Z) then (Z, Y) into the same accumulator
      for (int ps = 0; ps < passes; ++ps) {
        const uint32_t sA = (cls == 0 || ps == 0) ? sY : sZ;
        const uint32_t sB = (cls == 0 || ps == 1) ? sY : sZ;
        for (int kb = 0; kb < 2; ++kb) {
          const uint64_t dA0 = make_smem_desc_sw<128>(sA + kb * kBoxBytesS), dA1 = make_smem_desc_sw<128>(sA + kPlaneBytesS + kb * kBoxBytesS);
          const uint64_t dB0 = make_smem_desc_sw<128>(sB + kb * kBoxBytesS), dB1 = make_smem_desc_sw<128>(sB + kPlaneBytesS + kb * kBoxBytesS);
#pragma unroll
          for (int k = 0; k < kBoxK / 16; ++k) {
            const uint64_t ko = (uint64_t)(k * 2);
            umma_f16<1>(acc, dA1 + ko, dB0 + ko, IDESC, (ps | kb | k) ? 1u : 0u);     // lo * hi
            umma_f16<1, 1>(acc, dA0 + ko, dB1 + ko, IDESC, 1u);                        // hi * lo (A.hi kept in the collector)
            umma_f16<1, 2>(acc, dA0 + ko, dB0 + ko, IDESC, 1u);                        // hi * hi
          }
        }
      }
    }
    umma_commit<1>(smem_u32(&sh->bar_mma));
  };

  // The products of layer n + 1 need the planes of layer n but not the controller's decision (branch and coefficients
  // only enter the epilogue), so they are issued as soon as the planes are written and run under the reduction and
  // the controller of layer n.  When the controller stops, that last set of products was issued in vain.
  if (warp == kWarpIssue && elect_one()) issue_products();
  for (;;) {
    mbar_wait(smem_u32(&sh->bar_mma), mma_phase);
    mma_phase ^= 1u;
    tc_fence_after();

    // ---- epilogue of every class, in place
    const Sp2Coef& cf = ctrl->coef;
    double trs[1 + kMaxNbS], fros[1 + kMaxNbS], tracc = 0.0;
    float mxs[1 + kMaxNbS];
#pragma unroll
    for (int cls = 0; cls <= kMaxNbS; ++cls) {
      trs[cls] = 0.0; fros[cls] = 0.0; mxs[cls] = 0.f;
      if (cls > nb || !has_work) continue;
      uint8_t* Ph = smem + (size_t)(2 * cls) * kPlaneBytesS;
      uint8_t* Pm = Ph + kPlaneBytesS;
      const bool shift_row = cls == 0 && gi < n;            // zero padding stays zero
      const float a1hi = cls ? cf.a1z_hi[cls - 1] : cf.a1y_hi, a1lo = cls ? cf.a1z_lo[cls - 1] : cf.a1y_lo;
      const float a2 = cls ? cf.a2z[cls - 1] : cf.a2y;
      double unused = 0.0;
#pragma unroll
      for (int ch = 0; ch < 2; ++ch) {             // this warp's two 32-column chunks; the ones below the diagonal are skipped
        const int cidx = 2 * hh + ch, gj0 = cidx * 32;
        if (cidx < q) continue;
        small_epilogue(tmem_base + ((uint32_t)(q * 32) << 16) + (uint32_t)(cls * kNs + gj0), Ph, Pm, gi, gj0, lane, cidx == q, a1hi,
                       a1lo, a2, shift_row ? cf.dsh_hi : 0.f, shift_row ? cf.dsh_lo : 0.f, lo_round, lo_mask, trs[cls], fros[cls],
                       cls == 0 ? tracc : unused, mxs[cls]);
      }
    }
    // generic-proxy writes of the planes -> visible to the next layer's tcgen05.mma (async proxy)
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    tc_fence_before();

    // ---- per-warp partial sums of every class (fixed shuffle tree)
#pragma unroll
    for (int cls = 0; cls <= kMaxNbS; ++cls) {
      if (cls > nb) continue;
      double t = trs[cls], f = fros[cls], ta = tracc;
      float m = mxs[cls];
      if (has_work) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
          t += __shfl_xor_sync(0xffffffffu, t, o);
          f += __shfl_xor_sync(0xffffffffu, f, o);
          if (cls == 0) ta += __shfl_xor_sync(0xffffffffu, ta, o);
          const float qv = __shfl_xor_sync(0xffffffffu, m, o);
          m = (qv > m || qv != qv) ? qv : m;
        }
      }
      if (lane == 0) { sh->red[cls][0][warp] = t; sh->red[cls][1][warp] = f; sh->red[cls][2][warp] = ta; sh->redm[cls][warp] = m; }
    }
    __syncthreads();                               // planes written and fenced, accumulators read, partials in place
    if (warp == kWarpIssue && elect_one()) issue_products();     // layer n + 1, under the controller of layer n
    if (warp == 0) {
      // warp partials -> totals: lane w holds warp w's partial, fixed shuffle tree (deterministic); lane 0 then
      // fills the control block and runs the controller
      for (int cls = 0; cls <= nb; ++cls) {
        double t = lane < kWarpsS ? sh->red[cls][0][lane] : 0.0, f = lane < kWarpsS ? sh->red[cls][1][lane] : 0.0;
        double ta = (cls == 0 && lane < kWarpsS) ? sh->red[cls][2][lane] : 0.0;
        float mm = lane < kWarpsS ? sh->redm[cls][lane] : 0.f;
#pragma unroll
        for (int o = kWarpsS / 2; o > 0; o >>= 1) {
          t += __shfl_xor_sync(0xffffffffu, t, o);
          f += __shfl_xor_sync(0xffffffffu, f, o);
          if (cls == 0) ta += __shfl_xor_sync(0xffffffffu, ta, o);
          const float qv = __shfl_xor_sync(0xffffffffu, mm, o);
          mm = (qv > mm || qv != qv) ? qv : mm;
        }
        if (lane == 0) {
          if (cls == 0) {
            sp2_trace_identity(ctrl, ta);
            const double sy = sp2_exp2i(-ctrl->t);
            ctrl->tr_y = t * sy; ctrl->fro_y = f * sy * sy; ctrl->max_y = (double)mm * sy;
          } else {
            const double sz = sp2_exp2i(-ctrl->u[cls - 1]);
            ctrl->tr_z[cls - 1] = t * sz; ctrl->fro_z[cls - 1] = f * sz * sz; ctrl->max_z[cls - 1] = (double)mm * sz;
          }
        }
      }
      if (lane == 0) sp2_controller(ctrl);
    }
    __syncthreads();
    if (ctrl->done) {
      mbar_wait(smem_u32(&sh->bar_mma), mma_phase);   // the products issued in vain must retire before TMEM is released
      tc_fence_after();
      break;
    }
  }
}

// ---- the final planes (with their zero padding) and the control block go back to the workspace
__device__ __forceinline__ void small_store_state(const uint8_t* smem, const Sp2Ctrl* ctrl, const Sp2LayerArgs& a, int npad_g) {
  const int tid = threadIdx.x;
  const int par = ctrl->n & 1;                    // ping-pong buffer of the final iterate (what k_finalise and the hooks read)
  for (int p = 0; p < 2 + 2 * a.with_response; ++p) {
    __half* g = par ? a.out[p] : const_cast<__half*>(a.in[p]);
    const uint8_t* P = smem + (size_t)p * kPlaneBytesS;
    const int chunks_per_row = npad_g / 8;
    for (int idx = tid; idx < npad_g * chunks_per_row; idx += kThreadsS) {
      const int r = idx / chunks_per_row, c8 = idx % chunks_per_row;
      uint4 val = make_uint4(0u, 0u, 0u, 0u);
      if (r < kNs && c8 < kNs / 8) val = *reinterpret_cast<const uint4*>(P + sw_off(r, c8 * 8));
      *reinterpret_cast<uint4*>(g + (size_t)r * npad_g + c8 * 8) = val;
    }
  }
  const uint32_t* src = reinterpret_cast<const uint32_t*>(ctrl);
  uint32_t* dst = reinterpret_cast<uint32_t*>(a.ctrl);
  for (int i = tid; i < (int)(sizeof(Sp2Ctrl) / 4); i += kThreadsS) dst[i] = src[i];
}

// a: the argument block of layer parity 0 (tm[] / in[] = ping-pong buffer 0, which the prologue filled; out[] = buffer 1);
// npad_g: pitch of the global planes.
__global__ void __launch_bounds__(kThreadsS, 1) k_small_stack(const __grid_constant__ Sp2LayerArgs a, int npad_g) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~(uintptr_t)1023);
  const int nb = a.with_response;
  const int n_planes = 2 + 2 * nb;
  SmallShared* sh = reinterpret_cast<SmallShared*>(smem + (size_t)n_planes * kPlaneBytesS);
  Sp2Ctrl* ctrl = reinterpret_cast<Sp2Ctrl*>(sh->ctrl);
  const int tid = threadIdx.x, warp = tid >> 5;
  const uint32_t tmem_cols = nb == 0 ? 128u : (nb == 1 ? 256u : 512u);

  // ---- set-up: control block -> shared memory, barriers, TMEM, planes by TMA
  {
    const uint32_t* src = reinterpret_cast<const uint32_t*>(a.ctrl);
    uint32_t* dst = reinterpret_cast<uint32_t*>(ctrl);
    for (int i = tid; i < (int)(sizeof(Sp2Ctrl) / 4); i += kThreadsS) dst[i] = src[i];
  }
  if (tid == 0) {
    mbar_init(smem_u32(&sh->bar_load), 1);
    mbar_init(smem_u32(&sh->bar_mma), 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == kWarpAllocS) tmem_alloc<1>(smem_u32(&sh->tmem_base), tmem_cols);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *reinterpret_cast<volatile uint32_t*>(&sh->tmem_base);
  const bool active = ctrl->done == 0;
  if (active && tid == 0) {
    mbar_expect_tx(smem_u32(&sh->bar_load), (uint32_t)(n_planes * kPlaneBytesS));
    for (int p = 0; p < n_planes; ++p)
      for (int kb = 0; kb < 2; ++kb)
        tma_load_2d<1>(smem_u32(smem + (size_t)p * kPlaneBytesS + kb * kBoxBytesS), &a.tm[p], smem_u32(&sh->bar_load), kb * kBoxK, 0);
  }
  if (active) {
    mbar_wait(smem_u32(&sh->bar_load), 0);
    small_run_stack(smem, sh, ctrl, nb, a.n, a.lo_bits, tmem_base);
    small_store_state(smem, ctrl, a, npad_g);
  }
  tc_fence_before();
  __syncthreads();
  if (warp == kWarpAllocS) tmem_dealloc<1>(tmem_base, tmem_cols);
}

// ------------------------------------------------------------------------------------------
// The whole solve in one launch.  p: the problem (k_init's arguments), the caller's matrices, the ring entry.
template <typename TI, typename TO>
__global__ void __launch_bounds__(kThreadsS, 1) k_small_solve(const __grid_constant__ Sp2LayerArgs a, int npad_g,
                                                              const __grid_constant__ Sp2SmallProblem p) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~(uintptr_t)1023);
  const int nb = a.with_response;
  const int n_planes = 2 + 2 * nb;
  SmallShared* sh = reinterpret_cast<SmallShared*>(smem + (size_t)n_planes * kPlaneBytesS);
  Sp2Ctrl* ctrl = reinterpret_cast<Sp2Ctrl*>(sh->ctrl);
  const int tid = threadIdx.x, warp = tid >> 5;
  const uint32_t tmem_cols = nb == 0 ? 128u : (nb == 1 ? 256u : 512u);
  const int N = p.N;
  const TI* __restrict__ H = reinterpret_cast<const TI*>(p.H);

  // ---- control block (k_init), barriers, TMEM, zero planes
  {
    uint32_t* dst = reinterpret_cast<uint32_t*>(ctrl);
    for (int i = tid; i < (int)(sizeof(Sp2Ctrl) / 4); i += kThreadsS) dst[i] = 0u;
    uint4* pl = reinterpret_cast<uint4*>(smem);
    for (int i = tid; i < n_planes * kPlaneBytesS / 16; i += kThreadsS) pl[i] = make_uint4(0u, 0u, 0u, 0u);
  }
  if (tid == 0) {
    mbar_init(smem_u32(&sh->bar_mma), 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == kWarpAllocS) tmem_alloc<1>(smem_u32(&sh->tmem_base), tmem_cols);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *reinterpret_cast<volatile uint32_t*>(&sh->tmem_base);
  if (tid == 0) {
    ctrl->N = N; ctrl->n_occ = p.n_occ; ctrl->npad = npad_g; ctrl->with_response = nb;
    ctrl->max_layers = p.max_layers; ctrl->user_bounds = p.user_bounds; ctrl->user_eps_min = p.eps_min;
    ctrl->user_eps_max = p.eps_max; ctrl->tol = p.tol; ctrl->forced_layers = p.forced_layers;
    ctrl->forced_signs = p.forced_signs; ctrl->no_recentre = p.no_recentre;
  }

  // ---- a1: Gershgorin discs, tr H, max|H|, sum|H| (non-finite detector); two threads per row
  {
    const int row = tid >> 1, part = tid & 1;
    double s = 0.0, m = 0.0, d = 0.0;
    if (row < N) {
      const TI* r = H + (size_t)row * p.ldh;
      for (int j = part; j < N; j += 2) { const double v = fabs((double)r[j]); s += v; m = fmax(m, v); }
      d = (double)r[row];
    }
    s += __shfl_xor_sync(0xffffffffu, s, 1);
    m = fmax(m, __shfl_xor_sync(0xffffffffu, m, 1));
    const bool own = row < N && part == 0;
    const double rad = s - fabs(d);
    const double lo = block_min(own ? d - rad : INFINITY, sh, 0);
    const double hi = block_max(own ? d + rad : -INFINITY, sh, 1);
    const double tr = block_sum(own ? d : 0.0, sh, 2);
    const double mx = block_max(own ? m : 0.0, sh, 3);
    double sum = block_sum(own ? s : 0.0, sh, 4);
    for (int b = 0; b < nb; ++b) {                 // perturbations: max|H1_b| and the non-finite detector
      const TI* H1 = reinterpret_cast<const TI*>(p.H1[b]);
      double s1 = 0.0, m1 = 0.0;
      if (row < N) {
        const TI* r = H1 + (size_t)row * p.ldh;
        for (int j = part; j < N; j += 2) { const double v = fabs((double)r[j]); s1 += v; m1 = fmax(m1, v); }
      }
      const double mx1 = block_max(row < N ? m1 : 0.0, sh, 5);
      sum += block_sum(row < N ? s1 : 0.0, sh, 6);
      __syncthreads();                             // rows 5, 6 of red2 are reused by the next perturbation
      if (tid == 0) ctrl->maxabs_h1[b] = mx1;
    }
    __syncthreads();
    if (tid == 0) sp2_setup_input_layer(ctrl, lo, hi, tr, mx, sum, nb);
    __syncthreads();
  }

  if (!ctrl->done) {
    // ---- a2: Y_0 = X_0 - c_0 I, Z_0b = -H1_b / Delta, split into the planes in shared memory.  (H_ij + H_ji)/2 is
    // the same number for (i,j) and (j,i), so the planes are bit-symmetric; every element is visited once, which
    // counts the upper triangle twice in ||.||_F^2 as the controller expects.
    const double inv_delta = 1.0 / ctrl->delta;
    for (int cls = 0; cls <= nb; ++cls) {
      const TI* M = cls == 0 ? H : reinterpret_cast<const TI*>(p.H1[cls - 1]);
      uint8_t* Ph = smem + (size_t)(2 * cls) * kPlaneBytesS;
      uint8_t* Pm = Ph + kPlaneBytesS;
      const double shift = cls == 0 ? ctrl->tr_h / (double)N : 0.0;     // Y0_ii = (tr H / N - H_ii) / Delta
      const double scale = sp2_exp2i(cls == 0 ? ctrl->t : ctrl->u[cls - 1]);
      double tr = 0.0, fro = 0.0, mx = 0.0;
      for (int i = warp; i < N; i += kWarpsS)
      for (int j = (tid & 31); j < N; j += 32) {
        const double hsym = 0.5 * ((double)M[(size_t)i * p.ldh + j] + (double)M[(size_t)j * p.ldh + i]);
        const double v = ((i == j ? shift : 0.0) - hsym) * inv_delta * scale;
        const __half h = __float2half_rn((float)v);
        const __half m = __float2half_rn((float)(v - (double)__half2float(h)));
        const uint32_t o = sw_off(i, j);
        *reinterpret_cast<__half*>(Ph + o) = h;
        *reinterpret_cast<__half*>(Pm + o) = m;
        const double s = (double)(__half2float(h) + __half2float(m));
        fro += s * s;
        if (i == j) tr += s;
        mx = (fabs(s) > mx || s != s) ? fabs(s) : mx;
      }
      tr = block_sum(tr, sh, 0); fro = block_sum(fro, sh, 1); mx = block_max(mx, sh, 2);
      __syncthreads();
      if (tid == 0) {
        if (cls == 0) {
          const double sy = sp2_exp2i(-ctrl->t);
          ctrl->tr_y = tr * sy; ctrl->fro_y = fro * sy * sy; ctrl->max_y = mx * sy;
        } else {
          const double sz = sp2_exp2i(-ctrl->u[cls - 1]);
          ctrl->tr_z[cls - 1] = tr * sz; ctrl->fro_z[cls - 1] = fro * sz * sz; ctrl->max_z[cls - 1] = mx * sz;
        }
      }
    }
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");    // the planes are read by tcgen05.mma next
    __syncthreads();
    if (tid == 0) sp2_controller(ctrl);             // decision for layer 0 (k_ctrl0)
    __syncthreads();

    // ---- a3-a5
    if (!ctrl->done) small_run_stack(smem, sh, ctrl, nb, N, a.lo_bits, tmem_base);
  }

  // ---- a6: D = c I + Y 2^-t, D1_b = Z_b 2^-u_b in the caller's dtype; tr D, tr(DH), tr D1_b; result struct
  const int st = ctrl->status;
  const bool ok = ctrl->done && (st == SP2_OK || st == SP2_WARN_NOT_CONVERGED);
  double trd = 0.0, trdh = 0.0, trd1[kMaxNbS] = {0.0, 0.0};
  if (ok) {
    TO* __restrict__ D = reinterpret_cast<TO*>(p.D);
    const double sy = sp2_exp2i(-ctrl->t), shift = ctrl->c;
    for (int i = warp; i < N; i += kWarpsS)
    for (int j = (tid & 31); j < N; j += 32) {
      const uint32_t o = sw_off(i, j);
      const double y = (double)(__half2float(*reinterpret_cast<const __half*>(smem + o)) +
                                __half2float(*reinterpret_cast<const __half*>(smem + kPlaneBytesS + o))) * sy;
      const double x = y + (i == j ? shift : 0.0);
      D[(size_t)i * p.ldd + j] = (TO)x;
      trdh += x * (double)H[(size_t)i * p.ldh + j];
      if (i == j) trd += x;
      for (int b = 0; b < nb; ++b) {
        const uint8_t* Pz = smem + (size_t)(2 + 2 * b) * kPlaneBytesS;
        const double z = (double)(__half2float(*reinterpret_cast<const __half*>(Pz + o)) +
                                  __half2float(*reinterpret_cast<const __half*>(Pz + kPlaneBytesS + o))) * sp2_exp2i(-ctrl->u[b]);
        reinterpret_cast<TO*>(p.D1[b])[(size_t)i * p.ldd + j] = (TO)z;
        if (i == j) trd1[b] += z;
      }
    }
  }
  trd = block_sum(trd, sh, 0); trdh = block_sum(trdh, sh, 1);
  for (int b = 0; b < kMaxNbS; ++b) trd1[b] = block_sum(trd1[b], sh, 2 + b);
  __syncthreads();
  if (tid == 0) {
    ctrl->tr_d = trd; ctrl->tr_dh = trdh;
    for (int b = 0; b < nb; ++b) ctrl->tr_d1[b] = trd1[b];
    sp2_result_t r;
    r.status = ctrl->done ? st : SP2_INTERNAL_INCOMPLETE; r.layers = ctrl->n;
    r.sign_mask[0] = ctrl->sign_mask[0]; r.sign_mask[1] = ctrl->sign_mask[1];
    r.stop_reason = ctrl->stop_reason; r.reserved = 0;
    r.tr_d = trd; r.tr_dh = trdh; r.tr_d1 = trd1[0];
    r.idem_est = ok ? ctrl->e[ctrl->n] : 0.0;
    r.eps_min = ctrl->eps_min; r.eps_max = ctrl->eps_max; r.gpu_ms = 0.f; r.layers_ms = 0.f; r.kernel_launches = 0; r.bounds_fallback = 0;
    *p.ring_entry = r;
  }
  __syncthreads();
  small_store_state(smem, ctrl, a, npad_g);
  tc_fence_before();
  __syncthreads();
  if (warp == kWarpAllocS) tmem_dealloc<1>(tmem_base, tmem_cols);
}

}  // namespace

// ------------------------------------------------------------------------------------------
int sp2_small_max_n() { return kNs; }
int sp2_small_max_nb() { return kMaxNbS; }

static size_t small_smem_bytes(int nb) { return (size_t)(2 + 2 * nb) * kPlaneBytesS + sizeof(SmallShared) + 1024; }

cudaError_t sp2_small_configure() {
  const int smem = (int)small_smem_bytes(kMaxNbS);
  cudaError_t e = cudaFuncSetAttribute(k_small_stack, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
  if (e == cudaSuccess) e = cudaFuncSetAttribute(k_small_solve<float, float>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
  if (e == cudaSuccess) e = cudaFuncSetAttribute(k_small_solve<float, double>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
  if (e == cudaSuccess) e = cudaFuncSetAttribute(k_small_solve<double, float>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
  if (e == cudaSuccess) e = cudaFuncSetAttribute(k_small_solve<double, double>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
  return e;
}

// args0: the argument block whose tm[] / in[] describe ping-pong buffer 0 (what the prologue wrote) and whose out[]
// describe buffer 1; npad_g: pitch of the global planes.
cudaError_t sp2_launch_small(const Sp2LayerArgs& args0, int npad_g, cudaStream_t s) {
  k_small_stack<<<1, kThreadsS, small_smem_bytes(args0.with_response), s>>>(args0, npad_g);
  return cudaGetLastError();
}

// the whole solve (prologue, stack, finalise) of a small problem in one launch
cudaError_t sp2_launch_small_solve(const Sp2LayerArgs& args0, int npad_g, const Sp2SmallProblem& p, cudaStream_t s) {
  const size_t smem = small_smem_bytes(args0.with_response);
  if (p.in_f64 && p.out_f64) k_small_solve<double, double><<<1, kThreadsS, smem, s>>>(args0, npad_g, p);
  else if (p.in_f64) k_small_solve<double, float><<<1, kThreadsS, smem, s>>>(args0, npad_g, p);
  else if (p.out_f64) k_small_solve<float, double><<<1, kThreadsS, smem, s>>>(args0, npad_g, p);
  else k_small_solve<float, float><<<1, kThreadsS, smem, s>>>(args0, npad_g, p);
  return cudaGetLastError();
}

// ================================================================================================
// sp2_density_noalloc (include/sp2.h): the one-CTA solve for callers that may not allocate.
//
// k_small_solve keeps the iterate in shared memory, but it still has global scratch: the final hi/lo planes of both
// ping-pong buffers (small_store_state: what the handle's debug hooks and the refinement read), the control block
// and the result entry.  A handle carves those out of the caller's workspace; here they live in ONE file-scope device
// array that every GPU which loads the library holds until the process exits.  The kernel is the same k_small_solve
// (density only), the library options are the defaults, and the matrices are the caller's.
//
// In host code `g_noalloc_scratch` is a host-side stand-in for the symbol, NOT a device address: the address the kernel
// gets comes from cudaGetSymbolAddress, asked once per device with that device current.
namespace {

constexpr int kNoAllocMaxN = kNs;                                                  // 128
constexpr size_t kNoAllocPlaneBytes = (size_t)kNs * kNs * sizeof(__half);          // one global plane, pitch kNs
constexpr size_t kNoAllocCtrlOff = 4 * kNoAllocPlaneBytes;                         // Yh, Ym of buffers 0 and 1
constexpr size_t kNoAllocResultOff = kNoAllocCtrlOff + ((sizeof(Sp2Ctrl) + 255) / 256) * 256;
constexpr size_t kNoAllocBytes = kNoAllocResultOff + 256;

constexpr int kNoAllocMaxDevices = 64;
struct NoAllocDevice {
  int state;               // 0: not set up, 1: ready, < 0: -(sp2_status_t) of the failed set-up
  int cuda_error;
  unsigned char* scratch;  // DEVICE address of g_noalloc_scratch on this device
};
NoAllocDevice g_noalloc_dev[kNoAllocMaxDevices];
std::mutex g_noalloc_mutex;

}  // namespace

static __device__ __align__(256) unsigned char g_noalloc_scratch[kNoAllocBytes];
static_assert(kNoAllocBytes <= 160 * 1024, "sp2_density_noalloc: the static scratch is documented as <= 160 KB per GPU");
static_assert(sizeof(sp2_result_t) <= 256, "result entry");

namespace {

// once per device, with that device current: architecture check, shared-memory opt-in of the kernel, symbol address
sp2_status_t noalloc_setup(int dev, NoAllocDevice** out) {
  if (dev < 0 || dev >= kNoAllocMaxDevices) return SP2_ERR_INVALID_ARG;
  std::lock_guard<std::mutex> lock(g_noalloc_mutex);
  NoAllocDevice& d = g_noalloc_dev[dev];
  if (d.state == 0) {
    int major = 0;
    cudaError_t e = cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev);
    if (e != cudaSuccess) { d.state = -(int)SP2_ERR_CUDA; d.cuda_error = (int)e; }
    else if (major != 10) { d.state = -(int)SP2_ERR_ARCH; }
    else {
      e = sp2_small_configure();
      void* ptr = nullptr;
      if (e == cudaSuccess) e = cudaGetSymbolAddress(&ptr, g_noalloc_scratch);
      if (e != cudaSuccess || !ptr) { d.state = -(int)SP2_ERR_CUDA; d.cuda_error = (int)e; (void)cudaGetLastError(); }
      else { d.scratch = static_cast<unsigned char*>(ptr); d.state = 1; }
    }
  }
  if (d.state < 0) return (sp2_status_t)(-d.state);
  *out = &d;
  return SP2_OK;
}

}  // namespace

extern "C" size_t sp2_noalloc_scratch_bytes(void) { return kNoAllocBytes; }
extern "C" int sp2_noalloc_max_n(void) { return kNoAllocMaxN; }

extern "C" sp2_status_t sp2_density_noalloc(const void* dH, sp2_dtype_t in_dtype, long ldh, int N, int N_occ, double tol,
                                            void* dD, sp2_dtype_t out_dtype, long ldd, sp2_result_t* d_result,
                                            sp2_result_t* out, void* stream) {
  if (N > kNoAllocMaxN) return SP2_ERR_TOO_LARGE;                    // beyond the static scratch: use a handle
  if (!dH || !dD || N < 2 || N_occ < 1 || N_occ >= N || ldh < N || ldd < N) return SP2_ERR_INVALID_ARG;
  if ((in_dtype != SP2_F32 && in_dtype != SP2_F64) || (out_dtype != SP2_F32 && out_dtype != SP2_F64)) return SP2_ERR_INVALID_ARG;
  if (!(tol >= 0.0)) return SP2_ERR_INVALID_ARG;
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return SP2_ERR_CUDA;
  NoAllocDevice* d = nullptr;
  sp2_status_t st = noalloc_setup(dev, &d);
  if (st != SP2_OK) return st;
  cudaStream_t s = static_cast<cudaStream_t>(stream);

  // the argument block of layer parity 0, as a handle's prepare() fills it for a density-only problem of pitch kNs;
  // k_small_solve reads in[] / out[] (state write-back), ctrl, with_response and lo_bits only (no TMA descriptors)
  Sp2LayerArgs a;
  memset(&a, 0, sizeof(a));
  __half* planes = reinterpret_cast<__half*>(d->scratch);
  const size_t pe = kNoAllocPlaneBytes / sizeof(__half);
  a.in[0] = planes;           a.in[1] = planes + pe;                 // buffer 0: Yh, Ym
  a.out[0] = planes + 2 * pe; a.out[1] = planes + 3 * pe;            // buffer 1
  a.ctrl = reinterpret_cast<Sp2Ctrl*>(d->scratch + kNoAllocCtrlOff);
  a.lo_bits = 11;
  a.n = N; a.npad = kNs; a.with_response = 0;
  sp2_result_t* entry = d_result ? d_result : reinterpret_cast<sp2_result_t*>(d->scratch + kNoAllocResultOff);

  Sp2SmallProblem p;
  memset(&p, 0, sizeof(p));
  p.H = dH; p.D = dD; p.ldh = ldh; p.ldd = ldd;
  p.N = N; p.n_occ = N_occ; p.max_layers = 100; p.user_bounds = 0; p.tol = tol;
  p.in_f64 = in_dtype == SP2_F64; p.out_f64 = out_dtype == SP2_F64; p.ring_entry = entry;
  // Nothing in the scratch has to start at zero: the kernel builds its control block and planes in shared memory and
  // only WRITES the global copies, in full, at its end.  The array keeps the last call's contents in between.
  cudaError_t e = sp2_launch_small_solve(a, kNs, p, s);
  if (e != cudaSuccess) return SP2_ERR_CUDA;
  if (!out) return SP2_OK;                                           // asynchronous: the status is in *d_result
  e = cudaMemcpyAsync(out, entry, sizeof(sp2_result_t), cudaMemcpyDeviceToHost, s);
  if (e == cudaSuccess) e = cudaStreamSynchronize(s);
  if (e != cudaSuccess) return SP2_ERR_CUDA;
  out->kernel_launches = 1;
  return (sp2_status_t)out->status;
}
