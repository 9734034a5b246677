// sp2_small.cu -- the whole DNN-SP2 layer stack of a SMALL problem (N <= 128) in ONE launch of ONE CTA, with the
// iterate resident in shared memory ("N <= 256: whole problem in one CTA's smem, all layers in one
// launch").
//
// At this size a layer is ~1 us of tensor work; what the multi-CTA kernels pay per layer -- global-memory round
// trips for the planes, a grid-wide barrier, the cross-CTA reduction -- is ten times that.  Here nothing leaves the
// SM between layers:
//   planes   Yh, Ym (and Zh_b, Zm_b for up to two perturbations) live in shared memory in the K-major SWIZZLE_128B
//            layout tcgen05.mma reads (two 128-row x 64-k boxes per plane, loaded once by TMA from the planes the
//            prologue wrote), and are updated IN PLACE: a layer's MMAs have all retired before its epilogue
//            writes, and only the thread that owns an upper-triangle element ever reads its old value;
//   products tcgen05.mma 128x128x16 kind::f16, FP32 accumulators in TMEM (128 columns for Y^2, 128 more per
//            perturbation for Y Z_b + Z_b Y): the same three plane products per k-step as the large kernel
//            (Eq. 20-22: X = X^(0) + X^(1), the lo*lo term dropped); K = 128 is one accumulation
//            segment (24 MMAs, fewer than the 96 of the large kernel's segments: DESIGN.md "truncation bias");
//   epilogue tcgen05.ld -> registers -> update, hi/lo split, element (i,j) and its mirror (j,i) written to shared
//            memory (bit-symmetric planes), partial sums;
//   control  block-wide reduction of the partial sums, then thread 0 runs the SAME controller as every other path
//            (sp2_controller: trace rule, stop test, shift, exponents) on a shared-memory copy of the control block.
// At the end the planes go back to the ping-pong buffer the finalise pass expects (layers & 1).
#include <cuda.h>
#include "sp2_internal.cuh"
#include "sp2_layer.h"
#include "sp2_ptx.cuh"

namespace {
using namespace sp2ptx;

constexpr int kNs = 128;                        // padded dimension of the small path (one UMMA tile)
constexpr int kBoxK = 64;                       // k extent of a TMA box (= sp2_layer_box_k())
constexpr int kBoxBytesS = kNs * kBoxK * 2;     // 16 KB: 128 rows x 128 bytes
constexpr int kPlaneBytesS = 2 * kBoxBytesS;    // 32 KB: k-blocks 0 and 1
constexpr int kThreadsS = 256;                  // 8 warps: TMEM lane quarter = warp & 3, column half = warp >> 2
constexpr int kMaxNbS = 2;                      // perturbations: planes (2 + 2 nb) x 32 KB <= 192 KB, TMEM (1 + nb) x 128 <= 512

struct SmallShared {
  uint64_t bar_load, bar_mma;
  uint32_t tmem_base, pad;
  double red[1 + kMaxNbS][3][8];                // per class and warp: tr, fro, tracc
  float redm[1 + kMaxNbS][8];
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

// One product class of one layer for this thread's row gi and its 64 columns j0 .. j0 + 63: new values from the
// accumulators and the old planes, written in place (element and mirror), partial sums.
//   Ph, Pm: the class's hi / lo planes in shared memory.  shift: add the diagonal shift (Y class, real rows only).
__device__ __forceinline__ void small_epilogue(uint32_t tcol, uint8_t* Ph, uint8_t* Pm, int gi, int j0, int lane,
                                               float a1hi, float a1lo, float a2, float dsh_hi, float dsh_lo,
                                               uint32_t lo_round, uint32_t lo_mask,
                                               double& tr, double& fro, double& tracc, float& mxo) {
  float fsum = 0.f, mx = mxo, dval = 0.f, dacc = 0.f;
#pragma unroll
  for (int ch = 0; ch < 2; ++ch) {
    const int gj0 = j0 + 32 * ch;
    if (gj0 + 31 < (gi - lane)) continue;          // whole chunk below the diagonal (warp-uniform): mirrored by its transpose
    const bool diag = (gj0 == gi - lane);          // the chunk that holds this warp's 32 x 32 diagonal block
    uint32_t v[32];
    tmem_ld32(tcol + 32 * ch, v);
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
        // weights: above the diagonal twice (the mirror image), on it once, below it not at all (diagonal chunk only)
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
  }
  mxo = mx;
  fro += (double)fsum;
  tr += (double)dval;
  tracc += (double)dacc;
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
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  constexpr uint32_t IDESC = make_idesc(kNs, kNs);
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
  if (warp == 1) tmem_alloc<1>(smem_u32(&sh->tmem_base), tmem_cols);
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
  if (active) mbar_wait(smem_u32(&sh->bar_load), 0);

  const int q = warp & 3, hh = warp >> 2;
  const int gi = q * 32 + lane;                    // this thread's row = its TMEM lane
  const int j0 = hh * 64;                          // its 64 columns
  const int drop = 11 - a.lo_bits;
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
  if (active && warp == 0 && elect_one()) issue_products();
  while (active) {
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
      if (cls > nb) continue;
      uint8_t* Ph = smem + (size_t)(2 * cls) * kPlaneBytesS;
      uint8_t* Pm = Ph + kPlaneBytesS;
      const bool shift_row = cls == 0 && gi < a.n;          // zero padding stays zero
      const float a1hi = cls ? cf.a1z_hi[cls - 1] : cf.a1y_hi, a1lo = cls ? cf.a1z_lo[cls - 1] : cf.a1y_lo;
      const float a2 = cls ? cf.a2z[cls - 1] : cf.a2y;
      double unused = 0.0;
      small_epilogue(tmem_base + ((uint32_t)(q * 32) << 16) + (uint32_t)(cls * kNs + j0), Ph, Pm, gi, j0, lane, a1hi, a1lo, a2,
                     shift_row ? cf.dsh_hi : 0.f, shift_row ? cf.dsh_lo : 0.f, lo_round, lo_mask, trs[cls], fros[cls],
                     cls == 0 ? tracc : unused, mxs[cls]);
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
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) {
        t += __shfl_xor_sync(0xffffffffu, t, o);
        f += __shfl_xor_sync(0xffffffffu, f, o);
        if (cls == 0) ta += __shfl_xor_sync(0xffffffffu, ta, o);
        const float qv = __shfl_xor_sync(0xffffffffu, m, o);
        m = (qv > m || qv != qv) ? qv : m;
      }
      if (lane == 0) { sh->red[cls][0][warp] = t; sh->red[cls][1][warp] = f; sh->red[cls][2][warp] = ta; sh->redm[cls][warp] = m; }
    }
    __syncthreads();                               // planes written and fenced, accumulators read, partials in place
    if (warp == 0 && elect_one()) {
      issue_products();                            // layer n + 1 under the controller of layer n
      for (int cls = 0; cls <= nb; ++cls) {        // warp partials in index order: deterministic
        double t = 0.0, f = 0.0, ta = 0.0;
        float mm = 0.f;
        for (int w = 0; w < 8; ++w) {
          t += sh->red[cls][0][w]; f += sh->red[cls][1][w]; ta += sh->red[cls][2][w];
          const float o = sh->redm[cls][w];
          mm = (o > mm || o != o) ? o : mm;
        }
        if (cls == 0) {
          sp2_trace_identity(ctrl, ta);
          const double sy = sp2_exp2i(-ctrl->t);
          ctrl->tr_y = t * sy; ctrl->fro_y = f * sy * sy; ctrl->max_y = (double)mm * sy;
        } else {
          const double sz = sp2_exp2i(-ctrl->u[cls - 1]);
          ctrl->tr_z[cls - 1] = t * sz; ctrl->fro_z[cls - 1] = f * sz * sz; ctrl->max_z[cls - 1] = (double)mm * sz;
        }
      }
      sp2_controller(ctrl);
    }
    __syncthreads();
    if (ctrl->done) {
      mbar_wait(smem_u32(&sh->bar_mma), mma_phase);   // the products issued in vain must retire before TMEM is released
      tc_fence_after();
      break;
    }
  }

  // ---- the final iterate goes to the ping-pong buffer the finalise pass reads (layers & 1), with its zero padding
  if (active) {
    const int par = ctrl->n & 1;
    for (int p = 0; p < n_planes; ++p) {
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
  tc_fence_before();
  __syncthreads();
  if (warp == 1) tmem_dealloc<1>(tmem_base, tmem_cols);
}

}  // namespace

// ------------------------------------------------------------------------------------------
int sp2_small_max_n() { return kNs; }
int sp2_small_max_nb() { return kMaxNbS; }

static size_t small_smem_bytes(int nb) { return (size_t)(2 + 2 * nb) * kPlaneBytesS + sizeof(SmallShared) + 1024; }

cudaError_t sp2_small_configure() {
  return cudaFuncSetAttribute(k_small_stack, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)small_smem_bytes(kMaxNbS));
}

// args0: the argument block whose tm[] / in[] describe ping-pong buffer 0 (what the prologue wrote) and whose out[]
// describe buffer 1; npad_g: pitch of the global planes.
cudaError_t sp2_launch_small(const Sp2LayerArgs& args0, int npad_g, cudaStream_t s) {
  k_small_stack<<<1, kThreadsS, small_smem_bytes(args0.with_response), s>>>(args0, npad_g);
  return cudaGetLastError();
}
