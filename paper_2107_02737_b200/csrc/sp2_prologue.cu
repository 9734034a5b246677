// sp2_prologue.cu -- input layer of DNN-SP2 and the finalise pass (a6).
// All three are HBM-bound streaming kernels: coalesced row reads, warp-shuffle reductions, fp64
// accumulation, per-block slots reduced in fixed order (no float atomics -> deterministic).
//
//   a1  k_bounds     Gershgorin discs r_i = sum_{j!=i} |H_ij|, eps_min/max, tr H, max|H|
//   --  k_setup      reduce a1, Delta, c_0 = tr(X_0)/N, first plane exponents
//   a2  k_rescale    Y_0 = X_0 - c_0 I with X_0 = (eps_max I - H)/Delta, Z_0 = -H1/Delta, hi/lo FP16 split
//                    (PAPER.md:145 input layer; Eq. 20-21 dual representation)
//   --  k_ctrl0      reduce a2 partials, run the controller for layer 0
//   a6  k_finalise   D = c_L I + Y_L, D1 = Z_L in the caller's dtype, tr D, tr(DH), tr D1
#include "sp2_internal.cuh"

namespace {

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}
__device__ __forceinline__ double warp_max(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
  return v;
}

// 16-byte vector loads: float4 / double2
__device__ __forceinline__ void abs_acc(const float4& x, double& s, double& m, double& q) {
  const double a = fabs((double)x.x), b = fabs((double)x.y), c = fabs((double)x.z), d = fabs((double)x.w);
  s += (a + b) + (c + d);
  q += (a * a + b * b) + (c * c + d * d);
  m = fmax(m, fmax(fmax(a, b), fmax(c, d)));
}
__device__ __forceinline__ void abs_acc(const double2& x, double& s, double& m, double& q) {
  const double a = fabs(x.x), b = fabs(x.y);
  s += a + b;
  q += a * a + b * b;
  m = fmax(m, fmax(a, b));
}
template <typename T> struct Vec16;
template <> struct Vec16<float> { using type = float4; static constexpr int n = 4; };
template <> struct Vec16<double> { using type = double2; static constexpr int n = 2; };

// ------------------------------------------------------------------------------------------
// a1: one warp per row, 8 rows per 256-thread block.  mode 0: full Gershgorin; mode 1: only
// max|.| and the non-finite detector (used for H1).
template <typename T>
__global__ void __launch_bounds__(256) k_bounds(const T* __restrict__ H, long ld, int N, int mode,
                                                Sp2BoundSlot* __restrict__ slots) {
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int row = blockIdx.x * 8 + warp;
  double lo = INFINITY, hi = -INFINITY, tr = 0.0, mx = 0.0, sum = 0.0, sumsq = 0.0;
  if (row < N) {
    const T* r = H + (size_t)row * ld;
    double s = 0.0, m = 0.0, q = 0.0;
    const bool vec_ok = ((reinterpret_cast<uintptr_t>(r) & 15) == 0);
    int j0 = 0;
    if (vec_ok) {
      using V = typename Vec16<T>::type;
      constexpr int VN = Vec16<T>::n;
      const V* rv = reinterpret_cast<const V*>(r);
      const int nv = N / VN;
      for (int v = lane; v < nv; v += 32) abs_acc(__ldg(rv + v), s, m, q);
      j0 = nv * VN;
    }
    for (int j = j0 + lane; j < N; j += 32) {
      const double a = fabs((double)__ldg(r + j));
      s += a;
      q += a * a;
      m = fmax(m, a);
    }
    s = warp_sum(s);
    q = warp_sum(q);
    m = warp_max(m);
    const double d = (double)__ldg(r + row);
    const double rad = s - fabs(d);          // sum over j != i
    lo = d - rad; hi = d + rad; tr = d; mx = m; sum = s; sumsq = q;
  }
  __shared__ double sh[6][8];
  if (lane == 0) { sh[0][warp] = lo; sh[1][warp] = hi; sh[2][warp] = tr; sh[3][warp] = mx; sh[4][warp] = sum; sh[5][warp] = sumsq; }
  __syncthreads();
  if (threadIdx.x == 0) {
    Sp2BoundSlot o;
    o.lo = sh[0][0]; o.hi = sh[1][0]; o.tr = sh[2][0]; o.mx = sh[3][0]; o.sum = sh[4][0]; o.sumsq = sh[5][0];
    for (int w = 1; w < 8; ++w) {
      o.lo = fmin(o.lo, sh[0][w]); o.hi = fmax(o.hi, sh[1][w]);
      o.tr += sh[2][w]; o.mx = fmax(o.mx, sh[3][w]); o.sum += sh[4][w]; o.sumsq += sh[5][w];
    }
    (void)mode;
    slots[blockIdx.x] = o;
  }
}

// ------------------------------------------------------------------------------------------
// Reduce the bound slots, fix the input layer and the first plane exponents.  One block.
__global__ void __launch_bounds__(256) k_setup(Sp2Ctrl* c, const Sp2BoundSlot* sh_slots, int n_h,
                                               const Sp2BoundSlot* s1_slots, int n_h1) {
  __shared__ double red[6][256];
  const int tid = threadIdx.x;
  double lo = INFINITY, hi = -INFINITY, tr = 0.0, mx = 0.0, sum = 0.0, sum1 = 0.0, sumsq = 0.0;
  for (int i = tid; i < n_h; i += 256) {
    lo = fmin(lo, sh_slots[i].lo); hi = fmax(hi, sh_slots[i].hi);
    tr += sh_slots[i].tr; mx = fmax(mx, sh_slots[i].mx); sum += sh_slots[i].sum; sumsq += sh_slots[i].sumsq;
  }
  const int nb = n_h1 > 0 ? c->with_response : 0;     // s1_slots = nb arrays of n_h1 slots, one per perturbation
  double mx1[SP2_NB];
  for (int b = 0; b < SP2_NB; ++b) mx1[b] = 0.0;
  for (int b = 0; b < nb; ++b)
    for (int i = tid; i < n_h1; i += 256) {
      mx1[b] = fmax(mx1[b], s1_slots[(size_t)b * n_h1 + i].mx);
      sum1 += s1_slots[(size_t)b * n_h1 + i].sum;
    }
  red[0][tid] = lo; red[1][tid] = hi; red[2][tid] = tr; red[3][tid] = fmax(mx, 0.0); red[4][tid] = sum + sum1;
  red[5][tid] = sumsq;
  __syncthreads();
  for (int w = 128; w > 0; w >>= 1) {
    if (tid < w) {
      red[0][tid] = fmin(red[0][tid], red[0][tid + w]);
      red[1][tid] = fmax(red[1][tid], red[1][tid + w]);
      red[2][tid] += red[2][tid + w];
      red[3][tid] = fmax(red[3][tid], red[3][tid + w]);
      red[4][tid] += red[4][tid + w];
      red[5][tid] += red[5][tid + w];
    }
    __syncthreads();
  }
  __shared__ double red1[256];
  for (int b = 0; b < nb; ++b) {
    red1[tid] = mx1[b];
    __syncthreads();
    for (int w = 128; w > 0; w >>= 1) {
      if (tid < w) red1[tid] = fmax(red1[tid], red1[tid + w]);
      __syncthreads();
    }
    if (tid == 0) c->maxabs_h1[b] = red1[0];
    __syncthreads();
  }
  if (tid != 0) return;
  sp2_setup_input_layer(c, red[0][0], red[1][0], red[2][0], red[3][0], red[4][0], nb, red[5][0]);
}

// ------------------------------------------------------------------------------------------
// a2: 32x32 tile pairs (bi <= bj).  Each block reads H tile (bi,bj) and (bj,bi), forms the
// symmetrised value, and writes both mirror images of the hi/lo planes with coalesced rows, so
// the planes are bit-symmetric by construction.  which = 0: Y from H, 1 + b: Z_b from H1_b.
// Pads (rows/cols >= N up to npad) are written as zero.
template <typename T>
__global__ void __launch_bounds__(256) k_rescale(const T* __restrict__ H, long ld, const Sp2Ctrl* __restrict__ c,
                                                 int which, __half* __restrict__ Ph, __half* __restrict__ Pm,
                                                 int npad, Sp2Slot* __restrict__ slots) {
  if (c->done) return;
  __shared__ double t1[32][33];
  __shared__ double t2[32][33];
  const int nb = npad >> 5;
  // decode blockIdx.x -> (bi, bj), bi <= bj, row-major over the upper triangle:
  // row bi starts at bi*nb - bi*(bi-1)/2
  const long idx = blockIdx.x;
  int bi = (int)floor(((2.0 * nb + 1.0) - sqrt((2.0 * nb + 1.0) * (2.0 * nb + 1.0) - 8.0 * (double)idx)) * 0.5);
  bi = max(0, min(nb - 1, bi));
  while (bi > 0 && (long)bi * nb - (long)bi * (bi - 1) / 2 > idx) --bi;
  while ((long)(bi + 1) * nb - (long)(bi + 1) * bi / 2 <= idx) ++bi;
  const int bj = bi + (int)(idx - ((long)bi * nb - (long)bi * (bi - 1) / 2));
  const int N = c->N;
  const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;   // 32 x 8
  for (int r = ty; r < 32; r += 8) {
    const int gi = bi * 32 + r, gj = bj * 32 + tx;
    t1[r][tx] = (gi < N && gj < N) ? (double)__ldg(H + (size_t)gi * ld + gj) : 0.0;
    const int hi_ = bj * 32 + r, hj = bi * 32 + tx;
    t2[r][tx] = (hi_ < N && hj < N) ? (double)__ldg(H + (size_t)hi_ * ld + hj) : 0.0;
  }
  __syncthreads();
  const double inv_delta = 1.0 / c->delta;
  const double shift = which == 0 ? c->tr_h / (double)N : 0.0;   // Y0_ii = (tr H/N - H_ii)/Delta
  const double scale = sp2_exp2i(which == 0 ? c->t : c->u[which - 1]);
  double tr = 0.0, fro = 0.0;
  float mx = 0.f;
  for (int r = ty; r < 32; r += 8) {
    // upper image: element (gi, gj) = (bi*32 + r, bj*32 + tx)
    {
      const int gi = bi * 32 + r, gj = bj * 32 + tx;
      double v = 0.0;
      if (gi < N && gj < N) {
        const double hsym = 0.5 * (t1[r][tx] + t2[tx][r]);
        v = ((gi == gj ? shift : 0.0) - hsym) * inv_delta * scale;
      }
      const __half h = __float2half_rn((float)v);
      const __half m = __float2half_rn((float)(v - (double)__half2float(h)));
      Ph[(size_t)gi * npad + gj] = h;
      Pm[(size_t)gi * npad + gj] = m;
      const float s = __half2float(h) + __half2float(m);
      const double w = (gj > gi) ? 2.0 : (gj == gi ? 1.0 : 0.0);
      fro += w * (double)s * (double)s;
      if (gi == gj) tr += (double)s;
      if (gj >= gi) mx = fmaxf(mx, fabsf(s));
      if (s != s) mx = s;
    }
    // lower image: element (gi, gj) = (bj*32 + r, bi*32 + tx), only for off-diagonal tile pairs
    if (bi != bj) {
      const int gi = bj * 32 + r, gj = bi * 32 + tx;
      double v = 0.0;
      if (gi < N && gj < N) {
        const double hsym = 0.5 * (t1[tx][r] + t2[r][tx]);
        v = (0.0 - hsym) * inv_delta * scale;
      }
      const __half h = __float2half_rn((float)v);
      const __half m = __float2half_rn((float)(v - (double)__half2float(h)));
      Ph[(size_t)gi * npad + gj] = h;
      Pm[(size_t)gi * npad + gj] = m;
    }
  }
  // block reduce -> slot
  __shared__ double rs[2][8];
  __shared__ float rm[8];
  tr = warp_sum(tr); fro = warp_sum(fro);
  float mxx = mx;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    const float q = __shfl_xor_sync(0xffffffffu, mxx, o);
    mxx = (q > mxx || q != q) ? q : mxx;
  }
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  if (lane == 0) { rs[0][warp] = tr; rs[1][warp] = fro; rm[warp] = mxx; }
  __syncthreads();
  if (threadIdx.x == 0) {
    Sp2Slot o; o.tr = 0.0; o.fro = 0.0; o.tracc = 0.0; o.mx = 0.f; o.pad = 0.f;
    for (int w = 0; w < 8; ++w) {
      o.tr += rs[0][w]; o.fro += rs[1][w];
      o.mx = (rm[w] > o.mx || rm[w] != rm[w]) ? rm[w] : o.mx;
    }
    slots[blockIdx.x] = o;
  }
}

// Reduce the a2 partials into TRUE units and run the controller for layer 0.  One block.
__global__ void __launch_bounds__(256) k_ctrl0(Sp2Ctrl* c, const Sp2Slot* ys, const Sp2Slot* zs, int count) {
  if (c->done) return;
  __shared__ double red[4 * 256];
  double tr, fro, mx, unused;
  sp2_reduce_slots(ys, count, red, tr, fro, mx, unused);
  const int nbz = c->pw_phase ? 0 : c->with_response;   // the power phase carries no perturbation
  for (int b = 0; b < nbz; ++b) {       // zs = one slot array of `count` per perturbation
    double trz, froz, mxz;
    sp2_reduce_slots(zs + (size_t)b * count, count, red, trz, froz, mxz, unused);
    if (threadIdx.x == 0) {
      const double sz = sp2_exp2i(-c->u[b]);
      c->tr_z[b] = trz * sz; c->fro_z[b] = froz * sz * sz; c->max_z[b] = mxz * sz;
    }
  }
  if (threadIdx.x != 0) return;
  const double sy = sp2_exp2i(-c->t);
  c->tr_y = tr * sy; c->fro_y = fro * sy * sy; c->max_y = mx * sy;
  sp2_controller(c);
}

// ------------------------------------------------------------------------------------------
// a6: D = c I + (Yh+Ym) 2^-t, D1 = (Zh+Zm) 2^-u;  tr D, tr(DH), tr D1.  One warp per row.
// The final iterate lives in buffer (layers & 1); both candidates are passed.  Batched response: one launch
// per perturbation zb with that perturbation's planes; launches zb > 0 pass D = nullptr and only write D1_zb.
template <typename TI, typename TO>
__global__ void __launch_bounds__(256) k_finalise(const Sp2Ctrl* __restrict__ c,
                                                  const __half* __restrict__ Yh0, const __half* __restrict__ Ym0,
                                                  const __half* __restrict__ Yh1, const __half* __restrict__ Ym1,
                                                  const __half* __restrict__ Zh0, const __half* __restrict__ Zm0,
                                                  const __half* __restrict__ Zh1, const __half* __restrict__ Zm1,
                                                  int npad, const TI* __restrict__ H, long ldh,
                                                  TO* __restrict__ D, TO* __restrict__ D1, long ldo, int zb,
                                                  double* __restrict__ slots /* 3 per block */) {
  const int st = c->status;
  if (!c->done || (st != SP2_OK && st != SP2_WARN_NOT_CONVERGED)) return;
  const int N = c->N;
  const int par = c->n & 1;
  const __half* Yh = par ? Yh1 : Yh0;
  const __half* Ym = par ? Ym1 : Ym0;
  const __half* Zh = par ? Zh1 : Zh0;
  const __half* Zm = par ? Zm1 : Zm0;
  const bool resp = c->with_response && D1 != nullptr;
  const double sy = sp2_exp2i(-c->t), sz = sp2_exp2i(-c->u[zb]), shift = c->c;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int row = blockIdx.x * 8 + warp;
  double trd = 0.0, trdh = 0.0, trd1 = 0.0;
  if (row < N) {
    const __half2* yh = reinterpret_cast<const __half2*>(Yh + (size_t)row * npad);
    const __half2* ym = reinterpret_cast<const __half2*>(Ym + (size_t)row * npad);
    const __half2* zh = reinterpret_cast<const __half2*>(Zh + (size_t)row * npad);
    const __half2* zm = reinterpret_cast<const __half2*>(Zm + (size_t)row * npad);
    const TI* h = H + (size_t)row * ldh;
    TO* d = D ? D + (size_t)row * ldo : nullptr;
    TO* d1 = resp ? D1 + (size_t)row * ldo : nullptr;
    for (int j2 = lane; 2 * j2 < N; j2 += 32) {
      float2 a = make_float2(0.f, 0.f), b = a;
      if (d) { a = __half22float2(yh[j2]); b = __half22float2(ym[j2]); }
      float2 p = make_float2(0.f, 0.f), q = p;
      if (resp) { p = __half22float2(zh[j2]); q = __half22float2(zm[j2]); }
#pragma unroll
      for (int e = 0; e < 2; ++e) {
        const int j = 2 * j2 + e;
        if (j >= N) break;
        if (d) {
          const double y = (double)((e ? a.y : a.x) + (e ? b.y : b.x)) * sy;
          const double x = y + (j == row ? shift : 0.0);
          d[j] = (TO)x;
          trdh += x * (double)__ldg(h + j);
          if (j == row) trd += x;
        }
        if (resp) {
          const double z = (double)((e ? p.y : p.x) + (e ? q.y : q.x)) * sz;
          d1[j] = (TO)z;
          if (j == row) trd1 += z;
        }
      }
    }
  }
  trd = warp_sum(trd); trdh = warp_sum(trdh); trd1 = warp_sum(trd1);
  __shared__ double sh[3][8];
  if (lane == 0) { sh[0][warp] = trd; sh[1][warp] = trdh; sh[2][warp] = trd1; }
  __syncthreads();
  if (threadIdx.x == 0) {
    double a = 0, b = 0, e = 0;
    for (int w = 0; w < 8; ++w) { a += sh[0][w]; b += sh[1][w]; e += sh[2][w]; }
    slots[3 * blockIdx.x + 0] = a; slots[3 * blockIdx.x + 1] = b; slots[3 * blockIdx.x + 2] = e;
  }
}

__global__ void __launch_bounds__(256) k_finalise_reduce(Sp2Ctrl* c, const double* slots, int count,
                                                         sp2_result_t* ring_entry) {
  __shared__ double red[3][256];
  const int tid = threadIdx.x;
  double a = 0, b = 0, e = 0;
  const int st = c->done ? c->status : SP2_INTERNAL_INCOMPLETE;
  const bool ok = (st == SP2_OK || st == SP2_WARN_NOT_CONVERGED);
  if (ok)
    for (int i = tid; i < count; i += 256) { a += slots[3 * i]; b += slots[3 * i + 1]; e += slots[3 * i + 2]; }
  red[0][tid] = a; red[1][tid] = b; red[2][tid] = e;
  __syncthreads();
  for (int w = 128; w > 0; w >>= 1) {
    if (tid < w) { red[0][tid] += red[0][tid + w]; red[1][tid] += red[1][tid + w]; red[2][tid] += red[2][tid + w]; }
    __syncthreads();
  }
  // perturbations b > 0 of a batched response: their finalise launches left tr D1_b in slot arrays b * count ..
  for (int bb = 1; bb < c->with_response; ++bb) {
    __shared__ double redb[256];
    double eb = 0.0;
    if (ok) for (int i = tid; i < count; i += 256) eb += slots[3 * ((size_t)bb * count + i) + 2];
    redb[tid] = eb;
    __syncthreads();
    for (int w = 128; w > 0; w >>= 1) { if (tid < w) redb[tid] += redb[tid + w]; __syncthreads(); }
    if (tid == 0) c->tr_d1[bb] = redb[0];
    __syncthreads();
  }
  if (tid != 0) return;
  c->tr_d = red[0][0]; c->tr_dh = red[1][0]; c->tr_d1[0] = red[2][0];
  sp2_result_t r;
  r.status = st; r.layers = c->n; r.sign_mask[0] = c->sign_mask[0]; r.sign_mask[1] = c->sign_mask[1];
  r.stop_reason = c->stop_reason; r.reserved = 0;
  r.tr_d = c->tr_d; r.tr_dh = c->tr_dh; r.tr_d1 = c->tr_d1[0];
  r.idem_est = ok ? c->e[c->n] : 0.0;
  r.eps_min = c->eps_min; r.eps_max = c->eps_max; r.gpu_ms = 0.f; r.layers_ms = 0.f; r.kernel_launches = 0; r.bounds_fallback = 0;
  *ring_entry = r;
}

// ------------------------------------------------------------------------------------------
// Optional tighter spectral bounds: k steps of the Lanczos process on H with a fixed start
// vector; [theta_min - beta_k, theta_max + beta_k] (extreme Ritz values widened by the last residual norm, the
// usual "safe" bound) replaces the Gershgorin interval where it is tighter.  HBM-bound: k reads of H.
//   k_lz_init    v_0(i) = cos(0.7 i + 0.3), normalised
//   k_lz_matvec  w = H v          (one warp per row, float64 accumulation)
//   k_lz_step    alpha_j = w.v;  w -= alpha_j v + beta_j v_prev;  beta_{j+1} = |w|;  v_prev = v;  v = w / beta_{j+1}
//   k_lz_finish  extreme eigenvalues of T_k by Sturm bisection
__device__ inline double lz_block_sum(double v, double* sh /* 32 */) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  __syncthreads();
  if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = v;
  __syncthreads();
  double t = 0.0;
  for (int w = 0; w < (int)(blockDim.x >> 5); ++w) t += sh[w];
  return t;
}

__global__ void __launch_bounds__(1024) k_lz_init(Sp2Ctrl* c, int N, int steps, double* v, double* vprev) {
  __shared__ double sh[32];
  double s = 0.0;
  for (int i = threadIdx.x; i < N; i += 1024) { const double x = cos(0.7 * (double)i + 0.3); v[i] = x; vprev[i] = 0.0; s += x * x; }
  s = lz_block_sum(s, sh);
  const double inv = 1.0 / sqrt(s);
  for (int i = threadIdx.x; i < N; i += 1024) v[i] *= inv;
  if (threadIdx.x == 0) { c->lanczos_steps = steps; c->lz_beta[0] = 0.0; c->lz_min = NAN; c->lz_max = NAN; }
}

template <typename T>
__global__ void __launch_bounds__(256) k_lz_matvec(const T* __restrict__ H, long ld, int N, const double* __restrict__ v,
                                                   double* __restrict__ w) {
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int row = blockIdx.x * 8 + warp;
  if (row >= N) return;
  const T* r = H + (size_t)row * ld;
  double s = 0.0;
  for (int j = lane; j < N; j += 32) s += (double)__ldg(r + j) * v[j];
  s = warp_sum(s);
  if (lane == 0) w[row] = s;
}

__global__ void __launch_bounds__(1024) k_lz_step(Sp2Ctrl* c, int N, int j, double* v, double* vprev, double* w) {
  __shared__ double sh[32];
  const double beta = c->lz_beta[j];
  double a = 0.0;
  for (int i = threadIdx.x; i < N; i += 1024) a += w[i] * v[i];
  a = lz_block_sum(a, sh);
  double nn = 0.0;
  for (int i = threadIdx.x; i < N; i += 1024) {
    const double x = w[i] - a * v[i] - beta * vprev[i];
    w[i] = x;
    nn += x * x;
  }
  nn = lz_block_sum(nn, sh);
  const double bnew = sqrt(nn);
  const double inv = bnew > 0.0 ? 1.0 / bnew : 0.0;
  for (int i = threadIdx.x; i < N; i += 1024) { vprev[i] = v[i]; v[i] = w[i] * inv; }
  if (threadIdx.x == 0) { c->lz_alpha[j] = a; c->lz_beta[j + 1] = bnew; }
}

__global__ void k_lz_finish(Sp2Ctrl* c) {
  const int k = c->lanczos_steps;
  // eigenvalues of T_k lie in its own Gershgorin interval; count(x) = #eigenvalues < x by the Sturm recurrence
  double lo = INFINITY, hi = -INFINITY;
  for (int j = 0; j < k; ++j) {
    const double r = (j > 0 ? fabs(c->lz_beta[j]) : 0.0) + (j + 1 < k ? fabs(c->lz_beta[j + 1]) : 0.0);
    lo = fmin(lo, c->lz_alpha[j] - r);
    hi = fmax(hi, c->lz_alpha[j] + r);
  }
  auto count_below = [&](double x) {
    int cnt = 0;
    double d = 1.0;
    for (int j = 0; j < k; ++j) {
      const double b2 = j > 0 ? c->lz_beta[j] * c->lz_beta[j] : 0.0;
      d = (c->lz_alpha[j] - x) - (j > 0 ? b2 / d : 0.0);
      if (d == 0.0) d = -1e-300;
      if (d < 0.0) ++cnt;
    }
    return cnt;
  };
  double a = lo, b = hi;                 // smallest eigenvalue: count_below crosses from 0 to >= 1
  for (int it = 0; it < 200 && b - a > 1e-14 * fmax(fabs(a), fabs(b)); ++it) {
    const double m = 0.5 * (a + b);
    if (count_below(m) >= 1) b = m; else a = m;
  }
  const double th_min = a;
  a = lo; b = hi;                        // largest: count_below crosses from k-1 to k
  for (int it = 0; it < 200 && b - a > 1e-14 * fmax(fabs(a), fabs(b)); ++it) {
    const double m = 0.5 * (a + b);
    if (count_below(m) >= k) b = m; else a = m;
  }
  const double th_max = b;
  const double res = fabs(c->lz_beta[k]);
  c->lz_min = th_min - res;
  c->lz_max = th_max + res;
}

// ------------------------------------------------------------------------------------------
// Congruence transform support (sp2_congruence: H_orth = Z^T H Z, D = Z D_orth Z^T).
// k_gsetup: plane exponents from max|.| of the two inputs; k_split: matrix (or its transpose) -> hi/lo planes;
// k_gswap: operand exponents of the second product.
__global__ void __launch_bounds__(256) k_gsetup(Sp2Ctrl* c, const Sp2BoundSlot* sz, const Sp2BoundSlot* sa, int count, int N,
                                                sp2_result_t* ring_entry) {
  __shared__ double red[3][256];
  const int tid = threadIdx.x;
  double mz = 0.0, ma = 0.0, sum = 0.0;
  for (int i = tid; i < count; i += 256) { mz = fmax(mz, sz[i].mx); ma = fmax(ma, sa[i].mx); sum += sz[i].sum + sa[i].sum; }
  red[0][tid] = mz; red[1][tid] = ma; red[2][tid] = sum;
  __syncthreads();
  for (int w = 128; w > 0; w >>= 1) {
    if (tid < w) {
      red[0][tid] = fmax(red[0][tid], red[0][tid + w]);
      red[1][tid] = fmax(red[1][tid], red[1][tid + w]);
      red[2][tid] += red[2][tid + w];
    }
    __syncthreads();
  }
  if (tid != 0) return;
  const double maxz = red[0][0], maxa = red[1][0];
  c->g_el = sp2_pick_exponent(maxz);
  c->g_ex = sp2_pick_exponent(maxa);
  // |T_ij| = |sum_k L_ik A_jk| <= N max|L| max|A|: loose, but the lo plane keeps 2^-24 absolute resolution
  c->g_et = sp2_pick_exponent((double)N * maxz * maxa);
  c->g_ea = c->g_el; c->g_eb = c->g_ex;           // first product: A operand = L, B operand = X
  sp2_result_t r;
  memset(&r, 0, sizeof(r));
  r.status = isfinite(red[2][0]) ? SP2_OK : SP2_ERR_NONFINITE;
  *ring_entry = r;
}

__global__ void k_gswap(Sp2Ctrl* c) { c->g_ea = c->g_et; c->g_eb = c->g_el; }   // second product: T x L

template <typename T>
__global__ void __launch_bounds__(256) k_split(const T* __restrict__ A, long ld, int N, int npad, int transpose, int which,
                                               const Sp2Ctrl* __restrict__ c, __half* __restrict__ Ph, __half* __restrict__ Pm) {
  __shared__ double t[32][33];
  const int nb = npad >> 5;
  const int bi = blockIdx.x / nb, bj = blockIdx.x % nb;       // output tile (rows bi, cols bj)
  const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
  const double scale = sp2_exp2i(which == 0 ? c->g_el : c->g_ex);
  // source tile: rows (transpose ? bj : bi), cols (transpose ? bi : bj), read with coalesced rows
  for (int r = ty; r < 32; r += 8) {
    const int si = (transpose ? bj : bi) * 32 + r, sj = (transpose ? bi : bj) * 32 + tx;
    t[r][tx] = (si < N && sj < N) ? (double)__ldg(A + (size_t)si * ld + sj) : 0.0;
  }
  __syncthreads();
  for (int r = ty; r < 32; r += 8) {
    const double v = (transpose ? t[tx][r] : t[r][tx]) * scale;
    const float vf = (float)v;
    const __half hh = __float2half_rn(vf);
    const __half mm = __float2half_rn((float)(v - (double)__half2float(hh)));
    const size_t o = (size_t)(bi * 32 + r) * npad + bj * 32 + tx;
    Ph[o] = hh; Pm[o] = mm;
  }
}

// Trivial occupations (N_occ = 0 -> D = 0, N_occ = N -> D = I; D1 = 0), answered from the definition.
template <typename TO>
__global__ void __launch_bounds__(256) k_trivial(Sp2Ctrl* c, TO* __restrict__ D, TO* __restrict__ D1, long ldo,
                                                 sp2_result_t* ring_entry) {
  const int N = c->N;
  const double diag = (c->n_occ == 0) ? 0.0 : 1.0;
  for (size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x; idx < (size_t)N * N;
       idx += (size_t)gridDim.x * blockDim.x) {
    const int i = (int)(idx / N), j = (int)(idx % N);
    D[(size_t)i * ldo + j] = (TO)(i == j ? diag : 0.0);
    if (D1) D1[(size_t)i * ldo + j] = (TO)0.0;
  }
  if (blockIdx.x == 0 && threadIdx.x == 0) {
    const int st = c->status;   // k_setup may have flagged NONFINITE; DEGENERATE is fine here
    sp2_result_t r;
    r.status = (st == SP2_ERR_NONFINITE) ? st : SP2_OK;
    r.layers = 0; r.sign_mask[0] = r.sign_mask[1] = 0; r.stop_reason = 5; r.reserved = 0;
    r.tr_d = diag * N; r.tr_dh = diag * c->tr_h; r.tr_d1 = 0.0; r.idem_est = 0.0;
    r.eps_min = c->eps_min; r.eps_max = c->eps_max; r.gpu_ms = 0.f; r.layers_ms = 0.f; r.kernel_launches = 0; r.bounds_fallback = 0;
    *ring_entry = r;
  }
}

// Sequence steps enqueue a bounded number of layer launches and cannot top up without a host round trip: a stack
// that has not stopped by then is closed here (D is written from the iterate reached, as for max_layers).
__global__ void k_close(Sp2Ctrl* c) {
  if (c->done) return;
  c->done = 1; c->status = SP2_WARN_NOT_CONVERGED; c->stop_reason = 7;
}

// End of the power phase (sp2_options_t.power_squarings): the rigorous radius r = ||A^(2^s)||_F^(1/2^s) r0 from the
// Frobenius norm of the iterate the squarings left (PAPER.md:145 needs an interval that ENCLOSES the spectrum; this
// one does whatever the eigenvectors are: max_i |lambda_i - mu|^p <= tr (H - mu I)^p for even p).  The interval
// [mu - r, mu + r], widened by 1e-3 of r for the 22-bit arithmetic of the squarings and intersected with the
// Gershgorin discs, is handed to the regular solve as user bounds; the control block is reset for it.
__global__ void k_power_finish(Sp2Ctrl* c) {
  const int s = c->n;                               // squarings actually applied
  const bool have = c->pw_total > 0 && c->status == SP2_OK && c->fro_y > 0.0 && isfinite(c->fro_y);
  double lo = c->eps_min, hi = c->eps_max;          // Gershgorin (k_setup of the power phase kept it)
  if (have) {
    // ||A^(2^s)||_F = 2^pw_log2scale sqrt(fro_y);  r = r0 * that^(1/2^s)
    const double lg = (c->pw_log2scale + 0.5 * log2(c->fro_y)) / sp2_exp2i(s);
    const double r = c->pw_r0 * exp2(lg) * (1.0 + 1e-3);
    lo = fmax(lo, c->pw_mu - r);
    hi = fmin(hi, c->pw_mu + r);
  }
  const int keep_status = (c->status == SP2_ERR_NONFINITE) ? c->status : SP2_OK;
  c->pw_phase = 0;
  if (have && hi > lo) { c->user_bounds = 1; c->user_eps_min = lo; c->user_eps_max = hi; }
  c->n = 0; c->done = (keep_status != SP2_OK) ? 1 : 0; c->status = keep_status; c->stop_reason = 0;
  c->sign_mask[0] = 0ull; c->sign_mask[1] = 0ull;
  c->ticket = 0u; c->epoch = 0u;
  c->c = 0.0; c->t = 0; c->sigma_last = 0.0; c->fro_in = 0.0; c->t_in = 0;
}

__global__ void k_init(Sp2Ctrl* c, int N, int n_occ, int npad, int with_response, int max_layers,
                       int user_bounds, double eps_min, double eps_max, double tol,
                       int forced_layers, unsigned long long forced_signs, int no_recentre, int power_squarings) {
  // one thread: reset the whole control block
  Sp2Ctrl z;
  memset(&z, 0, sizeof(z));
  z.N = N; z.n_occ = n_occ; z.npad = npad; z.with_response = with_response;
  z.max_layers = max_layers; z.user_bounds = user_bounds; z.user_eps_min = eps_min; z.user_eps_max = eps_max;
  z.tol = tol; z.forced_layers = forced_layers; z.forced_signs = forced_signs; z.no_recentre = no_recentre;
  z.pw_total = power_squarings; z.pw_phase = power_squarings > 0 ? 1 : 0;
  *c = z;
}

}  // namespace

// ------------------------------------------------------------------------------------------
// host-side launchers (called from sp2_api.cu)
#define SP2_DISPATCH_IN(dt, CALL_F32, CALL_F64) \
  do { if ((dt) == SP2_F32) { CALL_F32; } else { CALL_F64; } } while (0)

void sp2_launch_init(Sp2Ctrl* c, int N, int n_occ, int npad, int with_response, int max_layers,
                     int user_bounds, double eps_min, double eps_max, double tol, int forced_layers,
                     unsigned long long forced_signs, int no_recentre, int power_squarings, cudaStream_t s) {
  k_init<<<1, 1, 0, s>>>(c, N, n_occ, npad, with_response, max_layers, user_bounds, eps_min, eps_max, tol,
                         forced_layers, forced_signs, no_recentre, power_squarings);
}

void sp2_launch_power_finish(Sp2Ctrl* c, cudaStream_t s) { k_power_finish<<<1, 1, 0, s>>>(c); }

void sp2_launch_close(Sp2Ctrl* c, cudaStream_t s) { k_close<<<1, 1, 0, s>>>(c); }

int sp2_bounds_blocks(int N) { return (N + 7) / 8; }

void sp2_launch_bounds(const void* H, sp2_dtype_t dt, long ld, int N, int mode, Sp2BoundSlot* slots, cudaStream_t s) {
  const int grid = sp2_bounds_blocks(N);
  SP2_DISPATCH_IN(dt, (k_bounds<float><<<grid, 256, 0, s>>>((const float*)H, ld, N, mode, slots)),
                  (k_bounds<double><<<grid, 256, 0, s>>>((const double*)H, ld, N, mode, slots)));
}

void sp2_launch_setup(Sp2Ctrl* c, const Sp2BoundSlot* sh, int n_h, const Sp2BoundSlot* s1, int n_h1, cudaStream_t s) {
  k_setup<<<1, 256, 0, s>>>(c, sh, n_h, s1, n_h1);
}

int sp2_rescale_blocks(int npad) { const int nb = npad / 32; return nb * (nb + 1) / 2; }

void sp2_launch_rescale(const void* H, sp2_dtype_t dt, long ld, const Sp2Ctrl* c, int which, __half* Ph, __half* Pm,
                        int npad, Sp2Slot* slots, cudaStream_t s) {
  const int grid = sp2_rescale_blocks(npad);
  SP2_DISPATCH_IN(dt, (k_rescale<float><<<grid, 256, 0, s>>>((const float*)H, ld, c, which, Ph, Pm, npad, slots)),
                  (k_rescale<double><<<grid, 256, 0, s>>>((const double*)H, ld, c, which, Ph, Pm, npad, slots)));
}

void sp2_launch_ctrl0(Sp2Ctrl* c, const Sp2Slot* ys, const Sp2Slot* zs, int count, cudaStream_t s) {
  k_ctrl0<<<1, 256, 0, s>>>(c, ys, zs, count);
}

int sp2_finalise_blocks(int N) { return (N + 7) / 8; }

// One launch for D (+ D1 of perturbation zb = 0, or none), or for D1_zb alone (D = nullptr, zb > 0).  planes[0..3] =
// Yh, Ym of buffers 0, 1; planes[4..7] = Zh, Zm of perturbation zb, buffers 0, 1.  slots: 3 * blocks doubles per zb.
void sp2_launch_finalise(Sp2Ctrl* c, __half* const planes[8], int npad, const void* H, sp2_dtype_t in_dt, long ldh,
                         void* D, void* D1, sp2_dtype_t out_dt, long ldo, int N, int zb, double* slots, cudaStream_t s) {
  const int grid = sp2_finalise_blocks(N);
  double* sl = slots + 3 * (size_t)grid * zb;
#define SP2_FIN(TI, TO)                                                                                     \
  k_finalise<TI, TO><<<grid, 256, 0, s>>>(c, planes[0], planes[1], planes[2], planes[3], planes[4], planes[5], \
                                          planes[6], planes[7], npad, (const TI*)H, ldh, (TO*)D, (TO*)D1, ldo, zb, sl)
  if (in_dt == SP2_F32 && out_dt == SP2_F32) SP2_FIN(float, float);
  else if (in_dt == SP2_F32 && out_dt == SP2_F64) SP2_FIN(float, double);
  else if (in_dt == SP2_F64 && out_dt == SP2_F32) SP2_FIN(double, float);
  else SP2_FIN(double, double);
#undef SP2_FIN
}

void sp2_launch_finalise_reduce(Sp2Ctrl* c, int N, double* slots, sp2_result_t* ring_entry, cudaStream_t s) {
  k_finalise_reduce<<<1, 256, 0, s>>>(c, slots, sp2_finalise_blocks(N), ring_entry);
}

void sp2_launch_trivial(Sp2Ctrl* c, void* D, void* D1, sp2_dtype_t out_dt, long ldo, int N,
                        sp2_result_t* ring_entry, cudaStream_t s) {
  const int grid = (int)(((size_t)N * N + 255) / 256 > 4096 ? 4096 : ((size_t)N * N + 255) / 256);
  if (out_dt == SP2_F32) k_trivial<float><<<grid, 256, 0, s>>>(c, (float*)D, (float*)D1, ldo, ring_entry);
  else k_trivial<double><<<grid, 256, 0, s>>>(c, (double*)D, (double*)D1, ldo, ring_entry);
}

void sp2_launch_gsetup(Sp2Ctrl* c, const Sp2BoundSlot* sz, const Sp2BoundSlot* sa, int count, int N, sp2_result_t* ring_entry,
                       cudaStream_t s) {
  k_gsetup<<<1, 256, 0, s>>>(c, sz, sa, count, N, ring_entry);
}
void sp2_launch_gswap(Sp2Ctrl* c, cudaStream_t s) { k_gswap<<<1, 1, 0, s>>>(c); }
void sp2_launch_split(const void* A, sp2_dtype_t dt, long ld, int N, int npad, int transpose, int which, const Sp2Ctrl* c,
                      __half* Ph, __half* Pm, cudaStream_t s) {
  const int nb = npad / 32;
  SP2_DISPATCH_IN(dt, (k_split<float><<<nb * nb, 256, 0, s>>>((const float*)A, ld, N, npad, transpose, which, c, Ph, Pm)),
                  (k_split<double><<<nb * nb, 256, 0, s>>>((const double*)A, ld, N, npad, transpose, which, c, Ph, Pm)));
}

void sp2_launch_lanczos(Sp2Ctrl* c, const void* H, sp2_dtype_t dt, long ld, int N, int steps, double* vecs, cudaStream_t s) {
  double* v = vecs; double* vprev = vecs + N; double* w = vecs + 2 * (size_t)N;
  k_lz_init<<<1, 1024, 0, s>>>(c, N, steps, v, vprev);
  for (int j = 0; j < steps; ++j) {
    SP2_DISPATCH_IN(dt, (k_lz_matvec<float><<<(N + 7) / 8, 256, 0, s>>>((const float*)H, ld, N, v, w)),
                    (k_lz_matvec<double><<<(N + 7) / 8, 256, 0, s>>>((const double*)H, ld, N, v, w)));
    k_lz_step<<<1, 1024, 0, s>>>(c, N, j, v, vprev, w);
  }
  k_lz_finish<<<1, 1, 0, s>>>(c);
}
