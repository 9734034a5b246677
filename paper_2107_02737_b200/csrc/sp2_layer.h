// sp2_layer.h -- launch interface of the layer kernels (sp2_layer.cu), used by sp2_api.cu.
#pragma once
#include <cuda.h>
#include <cuda_fp16.h>
#include <cuda_runtime.h>
#include "sp2_internal.cuh"

// Arguments of one layer launch.  tm[] are TMA descriptors of the INPUT planes (Yh, Ym, Zh, Zm):
// 2-D FP16 tensors npad x npad, box 64 (k) x 128 (rows), SWIZZLE_128B.
struct alignas(64) Sp2LayerArgs {
  CUtensorMap tm[4];
  const __half* in[4];   // the same input planes as raw pointers (epilogue reads the old tile)
  __half* out[4];        // output planes Yh', Ym', Zh', Zm' (the other ping-pong buffer)
  Sp2Ctrl* ctrl;
  Sp2Slot* slots;        // [z-class slots][y-class slots]
  const int2* tiles;     // (ti, tj), ti <= tj, upper-triangular tile list in L2-friendly order
  int n;                 // true dimension (rows/cols >= n are zero padding and stay zero)
  int npad;              // padded dimension (multiple of the tile edge)
  int n_tiles;           // number of upper-triangular tiles
  int with_response;
  int seg_kb;            // k-blocks (of 64) per in-TMEM accumulation segment; divides npad/64
};

size_t sp2_layer_smem_bytes();
int sp2_layer_slots(int npad, int cta_group, int with_response, int engine);
cudaError_t sp2_layer_configure();
cudaError_t sp2_launch_layer(const Sp2LayerArgs& args, int engine, int cta_group, int num_sms, cudaStream_t s);
