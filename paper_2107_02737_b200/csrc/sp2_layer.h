// sp2_layer.h -- launch interface of the layer kernels (sp2_layer.cu), used by sp2_api.cu.
#pragma once
#include <cuda.h>
#include <cuda_fp16.h>
#include <cuda_runtime.h>
#include "sp2_internal.cuh"

// One entry of a CTA(-pair)'s static work list: segments [seg0, seg1) of the k sweep(s) of `unit`.
// kind 0: the whole unit (accumulate, epilogue).  Units of the last, partial wave are cut along k so
// that every CTA(-pair) gets the same number of segments: kind 1 = contributor (accumulate, store the
// FP32 partial sums to scratch slot `slot`, bump flags[flag_id]); kind 2 = owner (accumulate, wait for
// `nparts` contributors, add their partials from slots slot..slot+nparts-1 in that order, epilogue).
struct Sp2Item {
  int unit, seg0, seg1, kind;
  int slot, nparts, flag_id, pad;
};

constexpr int kLockEvery = 16;   // k-blocks between two checkpoints of the producers' lockstep

// Arguments of one layer launch.  tm[] are TMA descriptors of the INPUT planes (Yh, Ym, then Zh, Zm of every
// perturbation b at 2 + 2b): 2-D FP16 tensors npad x npad, box sp2_layer_box_k() (k) x 128 (rows), swizzle = box row bytes.
#define SP2_LAYER_PLANES (2 + 2 * SP2_NB)
struct alignas(64) Sp2LayerArgs {
  CUtensorMap tm[SP2_LAYER_PLANES];
  const __half* in[SP2_LAYER_PLANES];   // the same input planes as raw pointers (epilogue reads the old tile)
  __half* out[SP2_LAYER_PLANES];        // output planes Yh', Ym', Zh', Zm', ... (the other ping-pong buffer)
  Sp2Ctrl* ctrl;
  Sp2Slot* slots;        // [z slots of perturbation 0] ... [z slots of perturbation nb - 1][y slots]
  const int2* tiles;     // (ti, tj), ti <= tj, upper-triangular tile list in L2-friendly order
  const Sp2Item* items;  // work lists of all CTA(-pair)s, concatenated
  const int* item_begin; // [n_clusters + 1] offsets into items
  float* scratch;        // split-k partial sums
  unsigned int* flags;   // one arrival counter per split unit (zero between launches)
  int n_flags;
  // soft lockstep of the TMA producers over the leading whole units of every work list; checkpoint counters
  // flags[n_flags .. n_flags + lock_kb / kLockEvery), zeroed with the split-k flags
  int lock_kb;           // k-blocks of the lockstep region (a multiple of kLockEvery, the same for every CTA; 0 = off)
  int lock_need;         // arrivals a producer waits for at a checkpoint (<= CTAs of the grid)
  int lock_polls;        // polls (256 ns apart) after which a producer gives the lockstep up for the rest of the launch
  int lo_bits;           // significant bits kept in the lo planes (11 = all)
  // plain-product mode (sp2_congruence): C = A B^T, A = tm[0..1], B = tm[2..3]
  int gemm_mode;         // 0: SP2 layer, 1: plain product
  int out_kind;          // 0: hi/lo planes out[0], out[1]; 1: float matrix cout; 2: double matrix cout
  void* cout;            // caller's output matrix (out_kind 1, 2)
  long ldc;
  int n_clusters;        // CTA(-pair)s the work lists were built for (= grid size / cta_group)
  int n;                 // true dimension (rows/cols >= n are zero padding and stay zero)
  int npad;              // padded dimension (multiple of the tile edge)
  int n_tiles;           // number of upper-triangular tiles
  int with_response;     // number of perturbations carried (0 .. SP2_NB)
  int seg_kb;            // k-blocks (of 64) per in-TMEM accumulation segment; divides npad/64
};

size_t sp2_layer_smem_bytes();
int sp2_layer_box_k();   // k extent of the TMA box (32: SWIZZLE_64B, 64: SWIZZLE_128B)
int sp2_layer_slots(int npad, int grid_ctas, int with_response, int engine);   // Sp2Slot entries one launch writes
cudaError_t sp2_layer_configure();
cudaError_t sp2_layer_max_coresident(int cta_group, int num_sms, int* out);
cudaError_t sp2_launch_layer(const Sp2LayerArgs& args, int engine, int cta_group, cudaStream_t s);
size_t sp2_layer_scratch_slot_bytes(int cta_group);
cudaError_t sp2_launch_layers_persistent(const Sp2LayerArgs* d_args, int cta_group, int grid_clusters, cudaStream_t s);

// sp2_small.cu: the whole stack of a small problem (N <= sp2_small_max_n(), at most sp2_small_max_nb() perturbations) in
// one launch of one CTA, iterate resident in shared memory.  args0 = the argument block of layer parity 0.
struct Sp2SmallProblem {   // everything k_small_solve needs beyond the plane pointers: k_init's arguments, the caller's matrices
  const void* H;
  const void* H1[2];
  void* D;
  void* D1[2];
  long ldh, ldd;
  int N, n_occ, max_layers, user_bounds;
  double eps_min, eps_max, tol;
  unsigned long long forced_signs;
  int forced_layers, no_recentre;
  int in_f64, out_f64;
  sp2_result_t* ring_entry;
};
int sp2_small_max_n();
int sp2_small_max_nb();
cudaError_t sp2_small_configure();
cudaError_t sp2_launch_small(const Sp2LayerArgs& args0, int npad_g, cudaStream_t s);
cudaError_t sp2_launch_small_solve(const Sp2LayerArgs& args0, int npad_g, const Sp2SmallProblem& p, cudaStream_t s);
