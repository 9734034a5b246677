// sp2_api.cu -- host side of the C ABI declared in include/sp2.h: workspace carving, TMA descriptor
// encoding, the launch sequence of one solve and result retrieval.
//
// One solve = k_init, k_bounds (H [, H1]), k_setup, k_rescale ([H1,] H), k_ctrl0,
//             max_layers x layer kernel (early-exit once the device controller sets `done`),
//             k_finalise, k_finalise_reduce   -- all on the caller's stream, no host round trip
// in between (the paper's design crosses to the CPU every layer).
#include <cuda.h>
#include <cudaTypedefs.h>
#include <cuda_runtime.h>
#include <new>
#include <stdio.h>
#include <string.h>
#include <utility>
#include <vector>

#include "sp2.h"
#include "sp2_internal.cuh"
#include "sp2_layer.h"

// launchers defined in sp2_prologue.cu
void sp2_launch_init(Sp2Ctrl* c, int N, int n_occ, int npad, int with_response, int max_layers, int user_bounds,
                     double eps_min, double eps_max, double tol, int forced_layers, unsigned long long forced_signs,
                     int no_recentre, int power_squarings, cudaStream_t s);
void sp2_launch_power_finish(Sp2Ctrl* c, cudaStream_t s);
int sp2_bounds_blocks(int N);
void sp2_launch_bounds(const void* H, sp2_dtype_t dt, long ld, int N, int mode, Sp2BoundSlot* slots, cudaStream_t s);
void sp2_launch_setup(Sp2Ctrl* c, const Sp2BoundSlot* sh, int n_h, const Sp2BoundSlot* s1, int n_h1, cudaStream_t s);
int sp2_rescale_blocks(int npad);
void sp2_launch_rescale(const void* H, sp2_dtype_t dt, long ld, const Sp2Ctrl* c, int which, __half* Ph, __half* Pm,
                        int npad, Sp2Slot* slots, cudaStream_t s);
void sp2_launch_ctrl0(Sp2Ctrl* c, const Sp2Slot* ys, const Sp2Slot* zs, int count, cudaStream_t s);
int sp2_finalise_blocks(int N);
void sp2_launch_finalise_reduce(Sp2Ctrl* c, int N, double* slots, sp2_result_t* ring_entry, cudaStream_t s);
void sp2_launch_finalise(Sp2Ctrl* c, __half* const planes[8], int npad, const void* H, sp2_dtype_t in_dt, long ldh,
                         void* D, void* D1, sp2_dtype_t out_dt, long ldo, int N, int zb, double* slots, cudaStream_t s);
void sp2_launch_trivial(Sp2Ctrl* c, void* D, void* D1, sp2_dtype_t out_dt, long ldo, int N, sp2_result_t* ring_entry,
                        cudaStream_t s);
void sp2_launch_gsetup(Sp2Ctrl* c, const Sp2BoundSlot* sz, const Sp2BoundSlot* sa, int count, int N, sp2_result_t* ring_entry,
                       cudaStream_t s);
void sp2_launch_gswap(Sp2Ctrl* c, cudaStream_t s);
void sp2_launch_split(const void* A, sp2_dtype_t dt, long ld, int N, int npad, int transpose, int which, const Sp2Ctrl* c,
                      __half* Ph, __half* Pm, cudaStream_t s);
void sp2_launch_close(Sp2Ctrl* c, cudaStream_t s);
void sp2_launch_lanczos(Sp2Ctrl* c, const void* H, sp2_dtype_t dt, long ld, int N, int steps, double* vecs, cudaStream_t s);
// sp2_refine.cu
cudaError_t sp2_refine_configure();
void sp2_refine_box(int* box_k, int* box_rows);
int sp2_refine_max_blocks();
size_t sp2_refine_parts_bytes(int blocks);
int sp2_refine_grid(int npad, int max_blocks);
int sp2_launch_refine(Sp2Ctrl* c, __half* const planes[4], int npad, int N, int n_layers, double* Xa, double* Xb,
                      const CUtensorMap* maps, double* slots, void* parts_region, int max_blocks, const void* H, sp2_dtype_t in_dt, long ldh, void* D,
                      sp2_dtype_t out_dt, long ldo, sp2_result_t* ring_entry, cudaStream_t s);

namespace {

constexpr int kRingCap = 4096;
constexpr int kPadTo = 256;          // npad is a multiple of the largest tile edge
constexpr int kSimtMaxN = 4096;
constexpr int kMaxClusters = 256;   // >= SM count of any sm_100 part
constexpr int kFlagWords = 2 * kMaxClusters + 32768;   // split-k flags, then the checkpoint counters of the producers' lockstep
constexpr int kSeqSlack = 8;        // extra layer launches per sequence step on top of the last finished step's count

inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }
inline int pad_n(int n) { return (int)align_up((size_t)n, kPadTo); }

// One carved region of the caller's workspace.  `used` is the extent (bytes from `off`) the calls made through the
// handle so far were entitled to write, computed from the launch geometry (NOT from the allocation formulas), so
// that tests can check used <= reserved and that nothing outside [off, off + used) was ever written
// (sp2_debug_layout; compute-sanitizer is not available on the GPU pool).
struct Region {
  char name[24];
  size_t off, reserved, used;
};

struct Layout {
  size_t plane_bytes;     // one FP16 plane at n_max
  int nb_max;             // perturbations the workspace has planes for (0: density only)
  size_t off_planes;      // 4 + 4 nb_max planes: [buf][Yh, Ym] then, per perturbation, [buf][Zh, Zm]
  size_t off_slots, slots_count;
  size_t off_slots2;      // second slot array (Z partials of the prologue)
  size_t off_bslots, bslots_count;
  size_t off_fslots;
  size_t off_tiles, tiles_count;
  size_t off_items, items_cap, off_item_begin, off_scratch, scratch_bytes, off_flags;
  size_t off_items_pw, items_pw_cap, off_item_begin_pw;
  size_t off_ctrl, off_ring, off_args;
  size_t off_staging, staging_each;
  size_t off_refine, refine_each, off_refine_slots, refine_slots_count, off_refine_parts;
  size_t off_lanczos;
  size_t total;
  std::vector<Region> regions;
  int r_plane0, r_slots, r_slots2, r_bslots, r_fslots, r_tiles, r_items, r_item_begin, r_items_pw, r_item_begin_pw, r_scratch, r_flags, r_ctrl, r_args, r_ring,
      r_staging0, r_lanczos, r_refine0, r_refine_slots, r_refine_parts;
};

int add_region(Layout& L, const char* name, size_t off, size_t reserved) {
  Region r;
  memset(&r, 0, sizeof(r));
  strncpy(r.name, name, sizeof(r.name) - 1);
  r.off = off; r.reserved = reserved; r.used = 0;
  L.regions.push_back(r);
  return (int)L.regions.size() - 1;
}

// float64 refinement: k_refine_expand writes 2 doubles per row (npad rows), k_refine_layer 2 per upper-triangular
// 128x128 tile, k_refine_finalise 1 per row
size_t refine_slot_doubles(size_t npad) {
  const size_t nb = npad / 128, grid = nb * (nb + 1) / 2;
  return 2 * (grid > npad ? grid : npad);
}

Layout make_layout(int n_max, int flags) {
  Layout L;
  L.regions.clear();
  const size_t npad = (size_t)pad_n(n_max);
  int resp = (flags >> 8) & 15;                      // SP2_WITH_BATCH(nb)
  if (resp > SP2_MAX_BATCH) resp = SP2_MAX_BATCH;
  if (resp == 0 && (flags & SP2_WITH_RESPONSE)) resp = 1;
  L.nb_max = resp;
  L.plane_bytes = align_up(npad * npad * 2, 1024);
  size_t off = 0;
  L.off_planes = off; off += L.plane_bytes * (4 + 4 * (size_t)resp);
  L.r_plane0 = (int)L.regions.size();
  for (int k = 0; k < 4 + 4 * resp; ++k) {
    char nm[24];
    snprintf(nm, sizeof(nm), "plane%d", k);
    add_region(L, nm, L.off_planes + (size_t)k * L.plane_bytes, L.plane_bytes);
  }
  // the layer kernel writes one slot per CTA and product class (grid <= kMaxClusters CTAs); the prologue's
  // k_rescale(H) and the SIMT scaffold use the same array with one slot per block
  size_t s_tc = (size_t)sp2_layer_slots((int)npad, kMaxClusters, resp, SP2_ENGINE_TCGEN05);
  size_t s_simt = npad <= (size_t)kSimtMaxN ? (size_t)sp2_layer_slots((int)npad, 0, resp, SP2_ENGINE_SIMT_DEBUG) : 0;
  size_t s_resc = (size_t)sp2_rescale_blocks((int)npad);
  L.slots_count = s_tc;
  if (s_simt > L.slots_count) L.slots_count = s_simt;
  if (s_resc > L.slots_count) L.slots_count = s_resc;
  auto carve = [&](const char* name, size_t bytes, size_t* off_out) {
    *off_out = off;
    const size_t reserved = align_up(bytes, 1024);
    const int id = add_region(L, name, off, reserved);
    off += reserved;
    return id;
  };
  L.r_slots = carve("slots", L.slots_count * sizeof(Sp2Slot), &L.off_slots);
  const size_t nb1 = resp > 1 ? (size_t)resp : 1;
  L.r_slots2 = carve("slots2", nb1 * s_resc * sizeof(Sp2Slot), &L.off_slots2);
  L.bslots_count = (size_t)sp2_bounds_blocks(n_max);
  L.r_bslots = carve("bslots", (1 + nb1) * L.bslots_count * sizeof(Sp2BoundSlot), &L.off_bslots);
  L.r_fslots = carve("fslots", 3 * nb1 * (size_t)sp2_finalise_blocks(n_max) * sizeof(double), &L.off_fslots);
  const size_t nt1 = npad / 128;
  L.tiles_count = nt1 * nt1;                 // the congruence products use every tile, the layers the upper triangle
  L.r_tiles = carve("tiles", L.tiles_count * sizeof(int2), &L.off_tiles);
  L.items_cap = (1 + nb1) * L.tiles_count + 1024;
  L.r_items = carve("items", L.items_cap * sizeof(Sp2Item), &L.off_items);
  L.r_item_begin = carve("item_begin", (kMaxClusters + 1) * sizeof(int), &L.off_item_begin);
  // density-only work lists for the power phase (sp2_options_t.power_squarings) of a solve that carries perturbations
  L.items_pw_cap = resp ? L.tiles_count + 1024 : 0;
  L.r_items_pw = carve("items_pw", L.items_pw_cap * sizeof(Sp2Item), &L.off_items_pw);
  L.r_item_begin_pw = carve("item_begin_pw", (resp ? (kMaxClusters + 1) : 0) * sizeof(int), &L.off_item_begin_pw);
  L.scratch_bytes = 2 * (size_t)kMaxClusters * sp2_layer_scratch_slot_bytes(1);
  if (2 * (size_t)(kMaxClusters / 2) * sp2_layer_scratch_slot_bytes(2) > L.scratch_bytes)
    L.scratch_bytes = 2 * (size_t)(kMaxClusters / 2) * sp2_layer_scratch_slot_bytes(2);
  L.r_scratch = carve("scratch", L.scratch_bytes, &L.off_scratch);
  L.r_flags = carve("flags", kFlagWords * sizeof(unsigned int), &L.off_flags);
  L.r_ctrl = carve("ctrl", sizeof(Sp2Ctrl), &L.off_ctrl);
  L.r_args = carve("args", 4 * sizeof(Sp2LayerArgs), &L.off_args);      // [0..1] the solve, [2..3] its power phase
  L.r_ring = carve("ring", (size_t)kRingCap * sizeof(sp2_result_t), &L.off_ring);
  L.r_staging0 = -1; L.staging_each = 0; L.off_staging = 0;
  if (flags & SP2_WITH_HOST_STAGING) {
    L.staging_each = align_up((size_t)n_max * (size_t)n_max * 8, 1024);
    L.off_staging = off;
    L.r_staging0 = (int)L.regions.size();
    for (int k = 0; k < (resp ? 4 : 2); ++k) {
      char nm[24];
      snprintf(nm, sizeof(nm), "staging%d", k);
      add_region(L, nm, off, L.staging_each);
      off += L.staging_each;
    }
  }
  L.r_lanczos = carve("lanczos", 3 * (size_t)n_max * sizeof(double), &L.off_lanczos);
  L.r_refine0 = -1; L.r_refine_slots = -1; L.r_refine_parts = -1; L.off_refine_parts = 0; L.refine_each = 0; L.off_refine = 0; L.off_refine_slots = 0;
  L.refine_slots_count = 0;
  if (flags & SP2_WITH_REFINEMENT) {
    L.refine_each = align_up(npad * npad * sizeof(double), 1024);
    L.off_refine = off;
    L.r_refine0 = add_region(L, "refine0", off, L.refine_each); off += L.refine_each;
    add_region(L, "refine1", off, L.refine_each); off += L.refine_each;
    L.refine_slots_count = refine_slot_doubles(npad);
    L.r_refine_slots = carve("refine_slots", L.refine_slots_count * sizeof(double), &L.off_refine_slots);
    L.r_refine_parts = carve("refine_parts", sp2_refine_parts_bytes(sp2_refine_max_blocks()), &L.off_refine_parts);
  }
  L.total = off;
  return L;
}

void default_options(sp2_options_t* o) {
  memset(o, 0, sizeof(*o));
  o->max_layers = 100;
  o->engine = SP2_ENGINE_TCGEN05;
  o->cta_group = 0;
}

}  // namespace

struct sp2_handle_s {
  int n_max, flags, device, num_sms;
  int nb_max;                    // perturbations the workspace can carry (0: density only)
  uint8_t* ws;
  size_t ws_bytes;
  Layout L;
  sp2_options_t opt;
  PFN_cuTensorMapEncodeTiled_v12000 encode;
  // per-(N, cta_group) cache
  int cur_n, cur_npad, cur_cg, cur_resp, cur_seg, cur_lo, cur_maxctas;
  int n_active;                  // CTA(-pair)s whose work list is not empty (grid of the persistent multi-layer launch)
  Sp2LayerArgs args[2];          // parity 0: buffer 0 -> 1, parity 1: buffer 1 -> 0
  Sp2LayerArgs args_pw[2];       // the same for the density-only power phase (= args when no perturbation is carried)
  int n_flags_pw, n_active_pw, cur_pw, cur_lock;
  std::vector<Sp2Item> items_pw_host;
  std::vector<int> item_begin_pw_host;
  std::vector<int2> tiles_host;
  std::vector<Sp2Item> items_host;
  std::vector<int> item_begin_host;
  int n_flags, n_clusters;
  int max_clusters[3];           // co-resident CTAs (cta_group 1) / CTA pairs (cta_group 2) of the layer kernel on this device
  cudaEvent_t ev0, ev1, evl0, evl1;
  int time_layers;               // record evl0/evl1 around the layer launches of the next solve
  sp2_result_t* h_result;        // pinned
  int last_cuda_error;
  int layers_hint;               // layers + slack of the last converged solve of the current shape (0 = unknown)
  int no_lanczos;                // this solve is the Gershgorin re-run after the device guard rejected the Lanczos bounds
  unsigned long long launches;
  // sequence state
  int seq_active, seq_N, seq_nocc, seq_steps;
  cudaEvent_t seq_ev[2];         // "step t finished" markers, polled (never waited on) by later steps
  double seq_tol;
  cudaStream_t seq_stream;

  __half* plane(int which /*0 Yh, 1 Ym, 2 + 2b Zh of perturbation b, 3 + 2b Zm*/, int buf) const {
    const int idx = (which < 2) ? (buf * 2 + which) : (4 + 4 * ((which - 2) >> 1) + buf * 2 + (which & 1));
    return reinterpret_cast<__half*>(ws + L.off_planes + (size_t)idx * L.plane_bytes);
  }
  Sp2Slot* slots() const { return reinterpret_cast<Sp2Slot*>(ws + L.off_slots); }
  Sp2Slot* slots2() const { return reinterpret_cast<Sp2Slot*>(ws + L.off_slots2); }   // nb arrays of sp2_rescale_blocks
  Sp2BoundSlot* bslots(int i) const { return reinterpret_cast<Sp2BoundSlot*>(ws + L.off_bslots) + (size_t)i * L.bslots_count; }
  double* fslots() const { return reinterpret_cast<double*>(ws + L.off_fslots); }
  int2* tiles() const { return reinterpret_cast<int2*>(ws + L.off_tiles); }
  Sp2Item* items() const { return reinterpret_cast<Sp2Item*>(ws + L.off_items); }
  Sp2Item* items_pw() const { return reinterpret_cast<Sp2Item*>(ws + L.off_items_pw); }
  int* item_begin_pw() const { return reinterpret_cast<int*>(ws + L.off_item_begin_pw); }
  int* item_begin() const { return reinterpret_cast<int*>(ws + L.off_item_begin); }
  float* scratch() const { return reinterpret_cast<float*>(ws + L.off_scratch); }
  unsigned int* split_flags() const { return reinterpret_cast<unsigned int*>(ws + L.off_flags); }
  Sp2Ctrl* ctrl() const { return reinterpret_cast<Sp2Ctrl*>(ws + L.off_ctrl); }
  Sp2LayerArgs* d_args() const { return reinterpret_cast<Sp2LayerArgs*>(ws + L.off_args); }   // copy of args[] for the persistent kernel
  sp2_result_t* ring() const { return reinterpret_cast<sp2_result_t*>(ws + L.off_ring); }
  void* staging(int i) const { return ws + L.off_staging + (size_t)i * L.staging_each; }
  double* lanczos_vecs() const { return reinterpret_cast<double*>(ws + L.off_lanczos); }
  double* refine_x(int i) const { return reinterpret_cast<double*>(ws + L.off_refine + (size_t)i * L.refine_each); }
  double* refine_slots() const { return reinterpret_cast<double*>(ws + L.off_refine_slots); }
  void* refine_parts() const { return ws + L.off_refine_parts; }
  // bookkeeping for sp2_debug_layout: this call may write [off, off + bytes) of region `id`
  void touch(int id, size_t bytes) {
    if (id >= 0 && id < (int)L.regions.size() && bytes > L.regions[id].used) L.regions[id].used = bytes;
  }
  void touch_plane(int which, int buf, size_t npad) {
    const int idx = (which < 2) ? (buf * 2 + which) : (4 + 4 * ((which - 2) >> 1) + buf * 2 + (which & 1));
    touch(L.r_plane0 + idx, npad * npad * 2);
  }
};

namespace {

#define SP2_CUDA(h, expr)                                   \
  do {                                                      \
    cudaError_t e_ = (expr);                                \
    if (e_ != cudaSuccess) { (h)->last_cuda_error = (int)e_; return SP2_ERR_CUDA; } \
  } while (0)

// Upper-triangular tile list in an L2-friendly order: G x G groups of tiles, so that the tiles that
// run concurrently (consecutive list entries) share row panels of the operand planes.  Consecutive groups share
// their ROW panels (same gi), so inside a group the tiles go column by column: a wave of CTA(-pair)s that
// straddles two groups then touches the next group's first columns only (1-2 new column panels instead of all G;
// measured: 14 % fewer DRAM reads than row by row).
void build_tiles(int nt, std::vector<int2>& out) {
  out.clear();
  const int G = 8;
  const int ng = (nt + G - 1) / G;
  for (int gi = 0; gi < ng; ++gi)
    for (int gj = gi; gj < ng; ++gj)
      for (int tj = gj * G; tj < (gj + 1) * G && tj < nt; ++tj)
        for (int ti = gi * G; ti < (gi + 1) * G && ti < nt; ++ti)
          if (tj >= ti) out.push_back(make_int2(ti, tj));
}

// Static work lists.  Units (first the 2-pass YZ+ZY units of every perturbation, then the Y^2
// units, each list in the L2-friendly tile order) are dealt whole to the least-loaded CTA(-pair) --
// equal costs make that a round-robin whose concurrent units are neighbours -- as long as they fit
// under T = ceil(total segments / clusters).  The units that do not fit (the last, partial wave) are cut
// along k into parts that fill every cluster up to T; the cluster holding the last part owns the
// epilogue.  Loads differ by at most one segment.
void build_schedule(int n_tiles, int resp, int segs_y, int nC, std::vector<Sp2Item>& items,
                    std::vector<int>& begin, int* n_flags, int* n_slots) {
  const int n_units = n_tiles * (1 + resp);          // resp = number of perturbations; their units come first
  auto cost = [&](int u) { return (u < resp * n_tiles) ? 2 * segs_y : segs_y; };
  long long total = 0;
  for (int u = 0; u < n_units; ++u) total += cost(u);
  const int T = (int)((total + nC - 1) / nC);
  std::vector<int> load(nC, 0);
  std::vector<std::vector<Sp2Item>> full(nC), contrib(nC), owner(nC);
  std::vector<int> leftover;
  for (int u = 0; u < n_units; ++u) {
    int best = 0;
    for (int c = 1; c < nC; ++c) if (load[c] < load[best]) best = c;
    if (load[best] + cost(u) <= T) {
      Sp2Item it = {u, 0, cost(u), 0, 0, 0, 0, 0};
      full[best].push_back(it);
      load[best] += cost(u);
    } else {
      leftover.push_back(u);
    }
  }
  int flags = 0, slots = 0;
  for (int u : leftover) {
    int pos = 0;
    const int cu = cost(u);
    std::vector<std::pair<int, Sp2Item>> parts;     // (cluster, item)
    while (pos < cu) {
      int best = 0;
      for (int c = 1; c < nC; ++c) if (T - load[c] > T - load[best]) best = c;
      int take = T - load[best];
      if (take <= 0) take = cu - pos;               // cannot happen (T * nC >= total); stay safe
      if (take > cu - pos) take = cu - pos;
      Sp2Item it = {u, pos, pos + take, 1, 0, 0, flags, 0};
      parts.push_back(std::make_pair(best, it));
      load[best] += take;
      pos += take;
    }
    const int np = (int)parts.size() - 1;            // contributors
    if (np == 0) {
      parts[0].second.kind = 0;
      full[parts[0].first].push_back(parts[0].second);
      continue;
    }
    for (int k = 0; k < np; ++k) {
      parts[k].second.slot = slots + k;
      contrib[parts[k].first].push_back(parts[k].second);
    }
    Sp2Item& own = parts[np].second;
    own.kind = 2; own.slot = slots; own.nparts = np;
    owner[parts[np].first].push_back(own);
    slots += np;
    ++flags;
  }
  items.clear();
  begin.assign(nC + 1, 0);
  for (int c = 0; c < nC; ++c) {
    begin[c] = (int)items.size();
    // contributors never wait, owners only wait for contributors: whole units, then contributors, then owners.
    // (Measured alternative: contributors first and owners early removes the 60-170 us an owner spends at the very
    // end waiting for its contributors, but staggers the CTAs from the start, so the panels they stream stop
    // coinciding in L2: 40 % more DRAM reads for the same layer time.  Kept: whole units first, in lockstep.)
    items.insert(items.end(), full[c].begin(), full[c].end());
    items.insert(items.end(), contrib[c].begin(), contrib[c].end());
    items.insert(items.end(), owner[c].begin(), owner[c].end());
  }
  begin[nC] = (int)items.size();
  *n_flags = flags;
  *n_slots = slots;
}

sp2_status_t encode_plane_map(sp2_handle_t h, CUtensorMap* map, const __half* base, int npad) {
  cuuint64_t gdim[2] = {(cuuint64_t)npad, (cuuint64_t)npad};
  cuuint64_t gstride[1] = {(cuuint64_t)npad * 2};
  const int bk = sp2_layer_box_k();
  cuuint32_t box[2] = {(cuuint32_t)bk, 128};
  cuuint32_t estr[2] = {1, 1};
  CUresult r = h->encode(map, CU_TENSOR_MAP_DATA_TYPE_FLOAT16, 2, const_cast<__half*>(base), gdim, gstride, box, estr,
                         CU_TENSOR_MAP_INTERLEAVE_NONE, bk == 64 ? CU_TENSOR_MAP_SWIZZLE_128B : CU_TENSOR_MAP_SWIZZLE_64B,
                         CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                         CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) { h->last_cuda_error = 100000 + (int)r; return SP2_ERR_CUDA; }
  return SP2_OK;
}

// Tile shape: CTA pairs on 256x256 tiles (cta_group::2) halve the operand traffic per flop and win at large N;
// single CTAs on 128x128 tiles have 4x more units to balance and less launch / cluster overhead and win below.
// Measured cross-over on B200 (round 2, back-to-back solves, us per layer cg1 / cg2): density N = 4096 224 / 260,
// 4608 300 / 288, 5120 424 / 426; with response N = 3072 281 / 281, 3584 434 / 415, 4096 636 / 568.
int pick_cta_group(sp2_handle_t h, int npad, int resp) {
  if (h->opt.cta_group == 1 || h->opt.cta_group == 2) return h->opt.cta_group;
  return npad >= (resp ? 3584 : 4608) ? 2 : 1;
}

// CTA(-pair)s of one layer launch: one per SM (pair of SMs), bounded by what the device can keep co-resident
// (sp2_create queried it): the split-k owners of the last wave wait for contributors, which must be running.
int layer_clusters(sp2_handle_t h, int cg) {
  int nC = h->num_sms / cg;
  if (nC > h->max_clusters[cg]) nC = h->max_clusters[cg];
  if (h->opt.max_ctas > 0 && nC > h->opt.max_ctas / cg) nC = h->opt.max_ctas / cg;
  if (nC > kMaxClusters / cg) nC = kMaxClusters / cg;
  return nC < 1 ? 1 : nC;
}

constexpr int kPersistMaxNpad = 2048;
constexpr int kLockstepMinNpad = 7168;

// (re)build the per-problem launch state: tile list, TMA descriptors, ping-pong argument blocks
sp2_status_t prepare(sp2_handle_t h, int N, int resp, cudaStream_t s) {
  const int npad = pad_n(N);
  const int cg = pick_cta_group(h, npad, resp);
  int seg = h->opt.seg_kb;
  // default: 4 k-blocks per in-TMEM segment; the residual truncation bias in tr D grows ~ N * segment length
  // (measured at 2/3 filling, the worst case: 3.8e-4 at N = 24000, 6.1e-4 at N = 32768 against the 1e-3 bar), so the
  // largest problems take shorter segments (1.5e-4 at N = 32768, at 15 % lower throughput) and problems up to
  // N = 8192 longer ones (8 k-blocks: 8e-5 at N = 8192, 2 % faster than 4)
  const bool seg_auto = seg != 1 && seg != 2 && seg != 4 && seg != 8 && seg != 16 && seg != 32;
  if (seg_auto) seg = npad > 24576 ? 2 : (npad > 8192 ? 4 : 8);
  while ((npad / 64) % seg) seg >>= 1;
  // Up to N = 2048 (the latency-bound, one-launch regime) the work lists are built at the granularity of a whole k sweep
  // and never cut a pass along k: the accumulation segments stay as above (they set the rounding error), but a unit
  // cut into three or four parts that are handed over through scratch one after the other is what made sizes whose
  // k-block count has no large power-of-two divisor slow (N = 1152: 9 segments of 2 k-blocks per sweep, 41 us per
  // density layer; N = 1664: 13 of 2, 73 us; N = 1024: 24 us).  Now 28 and 35 us.
  const bool small_regime = seg_auto && npad <= kPersistMaxNpad;
  const int segs_pass = (npad / 64) / seg;                 // accumulation segments per k sweep
  const int sched_segs = small_regime ? 1 : segs_pass;     // granularity of the work lists
  if (h->cur_n == N && h->cur_npad == npad && h->cur_cg == cg && h->cur_resp == resp && h->cur_seg == seg &&
      h->cur_lo == h->opt.lo_bits && h->cur_maxctas == h->opt.max_ctas && h->cur_pw == (h->opt.power_squarings > 0) &&
      h->cur_lock == h->opt.lockstep)
    return SP2_OK;
  const int nt = npad / (128 * cg);
  build_tiles(nt, h->tiles_host);
  SP2_CUDA(h, cudaMemcpyAsync(h->tiles(), h->tiles_host.data(), h->tiles_host.size() * sizeof(int2),
                              cudaMemcpyHostToDevice, s));
  const int nC = layer_clusters(h, cg);
  // (fewer units than CTA(-pair)s is fine: the schedule splits them along k, every SM gets work)
  int n_slots = 0;
  build_schedule((int)h->tiles_host.size(), resp, sched_segs, nC, h->items_host, h->item_begin_host,
                 &h->n_flags, &n_slots);
  if (sched_segs != segs_pass)
    for (Sp2Item& it : h->items_host) { it.seg0 *= segs_pass; it.seg1 *= segs_pass; }
  h->n_clusters = nC;
  h->n_active = 1;
  for (int c = 0; c < nC; ++c) if (h->item_begin_host[c + 1] > h->item_begin_host[c]) h->n_active = c + 1;
  if (h->items_host.size() > h->L.items_cap || h->tiles_host.size() > h->L.tiles_count ||
      (size_t)n_slots * sp2_layer_scratch_slot_bytes(cg) > h->L.scratch_bytes || h->n_flags > 2 * kMaxClusters ||
      (size_t)sp2_layer_slots(npad, cg * nC, resp, SP2_ENGINE_TCGEN05) > h->L.slots_count)
    return SP2_ERR_WORKSPACE;
  h->touch(h->L.r_tiles, h->tiles_host.size() * sizeof(int2));
  h->touch(h->L.r_items, h->items_host.size() * sizeof(Sp2Item));
  h->touch(h->L.r_item_begin, h->item_begin_host.size() * sizeof(int));
  h->touch(h->L.r_flags, kFlagWords * sizeof(unsigned int));
  h->touch(h->L.r_scratch, (size_t)n_slots * sp2_layer_scratch_slot_bytes(cg));
  SP2_CUDA(h, cudaMemcpyAsync(h->items(), h->items_host.data(), h->items_host.size() * sizeof(Sp2Item),
                              cudaMemcpyHostToDevice, s));
  SP2_CUDA(h, cudaMemcpyAsync(h->item_begin(), h->item_begin_host.data(), h->item_begin_host.size() * sizeof(int),
                              cudaMemcpyHostToDevice, s));
  SP2_CUDA(h, cudaMemsetAsync(h->split_flags(), 0, kFlagWords * sizeof(unsigned int), s));
  // power phase of a solve that carries perturbations: the same tiles, density-only work lists of their own
  const bool pw_lists = h->opt.power_squarings > 0 && resp > 0;
  h->n_flags_pw = h->n_flags; h->n_active_pw = h->n_active;
  if (pw_lists) {
    int n_slots_pw = 0;
    build_schedule((int)h->tiles_host.size(), 0, sched_segs, nC, h->items_pw_host, h->item_begin_pw_host,
                   &h->n_flags_pw, &n_slots_pw);
    if (sched_segs != segs_pass)
      for (Sp2Item& it : h->items_pw_host) { it.seg0 *= segs_pass; it.seg1 *= segs_pass; }
    h->n_active_pw = 1;
    for (int c = 0; c < nC; ++c) if (h->item_begin_pw_host[c + 1] > h->item_begin_pw_host[c]) h->n_active_pw = c + 1;
    if (h->items_pw_host.size() > h->L.items_pw_cap || (size_t)n_slots_pw * sp2_layer_scratch_slot_bytes(cg) > h->L.scratch_bytes ||
        h->n_flags_pw > 2 * kMaxClusters)
      return SP2_ERR_WORKSPACE;
    h->touch(h->L.r_items_pw, h->items_pw_host.size() * sizeof(Sp2Item));
    h->touch(h->L.r_item_begin_pw, h->item_begin_pw_host.size() * sizeof(int));
    h->touch(h->L.r_scratch, (size_t)n_slots_pw * sp2_layer_scratch_slot_bytes(cg));
    SP2_CUDA(h, cudaMemcpyAsync(h->items_pw(), h->items_pw_host.data(), h->items_pw_host.size() * sizeof(Sp2Item),
                                cudaMemcpyHostToDevice, s));
    SP2_CUDA(h, cudaMemcpyAsync(h->item_begin_pw(), h->item_begin_pw_host.data(), h->item_begin_pw_host.size() * sizeof(int),
                                cudaMemcpyHostToDevice, s));
  }
  SP2_CUDA(h, cudaStreamSynchronize(s));     // host vectors may be rebuilt by the next prepare
  // soft lockstep of the producers over the leading whole units every CTA(-pair) has (launch-per-layer mode only).
  // On by default from N = 7168: measured per-layer gain 2-3 % at N = 8192 with response (density-only unchanged),
  // 9 % at N = 12288, 11 % (D + D1) and 4 % (density) at N = 16384; no gain below.
  int lock_kb = 0;
  const bool lock_on = h->opt.lockstep == 1 || (h->opt.lockstep == 0 && npad >= kLockstepMinNpad);
  if (lock_on && npad > kPersistMaxNpad && h->n_active == nC) {
    lock_kb = 1 << 30;
    for (int c = 0; c < nC; ++c) {
      int whole = 0;
      for (int i = h->item_begin_host[c]; i < h->item_begin_host[c + 1] && h->items_host[i].kind == 0; ++i)
        whole += (h->items_host[i].seg1 - h->items_host[i].seg0) * seg;
      if (whole < lock_kb) lock_kb = whole;
    }
    lock_kb -= lock_kb % kLockEvery;
    const int room = (kFlagWords - h->n_flags) * kLockEvery;   // beyond it the producers free-run
    if (lock_kb > room) lock_kb = room;
  }
  for (int par = 0; par < 2; ++par) {
    Sp2LayerArgs& a = h->args[par];
    memset(&a, 0, sizeof(a));
    for (int w = 0; w < 2 + 2 * (resp > 1 ? resp : 1); ++w) {
      const bool have = (w < 2) || (w < 2 + 2 * h->nb_max);
      const __half* in = have ? h->plane(w, par) : h->plane(w & 1, par);
      __half* out = have ? h->plane(w, par ^ 1) : h->plane(w & 1, par ^ 1);
      a.in[w] = in; a.out[w] = out;
      sp2_status_t st = encode_plane_map(h, &a.tm[w], in, npad);
      if (st != SP2_OK) return st;
    }
    a.ctrl = h->ctrl(); a.slots = h->slots(); a.tiles = h->tiles();
    a.items = h->items(); a.item_begin = h->item_begin(); a.scratch = h->scratch(); a.flags = h->split_flags();
    a.n_flags = h->n_flags; a.n_clusters = h->n_clusters;
    a.lock_kb = lock_kb; a.lock_need = (cg * nC * 7) / 8;
    a.lock_polls = 16 + npad / 64;             // ~ half the duration of a whole unit (k-blocks x 1.2 us at the capped clock)
    a.lo_bits = (h->opt.lo_bits >= 6 && h->opt.lo_bits <= 10) ? h->opt.lo_bits : 11;
    a.n = N; a.npad = npad; a.n_tiles = (int)h->tiles_host.size(); a.with_response = resp; a.seg_kb = seg;
    Sp2LayerArgs& q = h->args_pw[par];          // the power phase: Y planes only
    q = a;
    q.with_response = 0;
    if (pw_lists) { q.items = h->items_pw(); q.item_begin = h->item_begin_pw(); q.n_flags = h->n_flags_pw; q.lock_kb = 0; }
  }
  SP2_CUDA(h, cudaMemcpyAsync(h->d_args(), h->args, 2 * sizeof(Sp2LayerArgs), cudaMemcpyHostToDevice, s));
  SP2_CUDA(h, cudaMemcpyAsync(h->d_args() + 2, h->args_pw, 2 * sizeof(Sp2LayerArgs), cudaMemcpyHostToDevice, s));
  SP2_CUDA(h, cudaStreamSynchronize(s));
  h->touch(h->L.r_args, 4 * sizeof(Sp2LayerArgs));
  h->layers_hint = 0;
  h->cur_n = N; h->cur_npad = npad; h->cur_cg = cg; h->cur_resp = resp; h->cur_seg = seg; h->cur_lo = h->opt.lo_bits;
  h->cur_maxctas = h->opt.max_ctas; h->cur_pw = h->opt.power_squarings > 0; h->cur_lock = h->opt.lockstep;
  return SP2_OK;
}

// the perturbations of one solve (device pointers, or host pointers for the *_host twins)
struct Pert {
  int nb;
  const void* H1[SP2_MAX_BATCH];
  void* D1[SP2_MAX_BATCH];
};

Pert make_pert(const void* H1, void* D1) {
  Pert P;
  memset(&P, 0, sizeof(P));
  if (H1 || D1) { P.nb = 1; P.H1[0] = H1; P.D1[0] = D1; }
  return P;
}

sp2_status_t check_args(sp2_handle_t h, const void* H, const Pert& P, sp2_dtype_t in_dt, long ldh, int N,
                        int N_occ, void* D, sp2_dtype_t out_dt, long ldd) {
  if (!h) return SP2_ERR_INVALID_ARG;
  if (!H || !D) return SP2_ERR_INVALID_ARG;
  if (P.nb < 0 || P.nb > SP2_MAX_BATCH) return SP2_ERR_INVALID_ARG;
  for (int b = 0; b < P.nb; ++b) if (!P.H1[b] || !P.D1[b]) return SP2_ERR_INVALID_ARG;
  if (P.nb > h->nb_max) return P.nb > 1 && h->nb_max > 0 ? SP2_ERR_WORKSPACE : SP2_ERR_INVALID_ARG;
  if (N <= 0 || N > h->n_max) return SP2_ERR_INVALID_ARG;
  if (N_occ < 0 || N_occ > N) return SP2_ERR_INVALID_ARG;
  if (ldh < N || ldd < N) return SP2_ERR_INVALID_ARG;
  if ((in_dt != SP2_F32 && in_dt != SP2_F64) || (out_dt != SP2_F32 && out_dt != SP2_F64)) return SP2_ERR_INVALID_ARG;
  if (h->opt.engine == SP2_ENGINE_SIMT_DEBUG && pad_n(N) > kSimtMaxN) return SP2_ERR_INVALID_ARG;
  if (h->opt.refine_layers > 0 && !(h->flags & SP2_WITH_REFINEMENT)) return SP2_ERR_WORKSPACE;
  return SP2_OK;
}

// One persistent launch for the whole stack?  Small problems: a layer is shorter than a launch and its tail.
// The smallest problems: one CTA, iterate resident in shared memory (sp2_small.cu).  Automatic choice only.
bool use_small(sp2_handle_t h) {
  return h->opt.engine == SP2_ENGINE_TCGEN05 && h->opt.persistent == 0 && h->cur_n <= sp2_small_max_n() &&
         h->cur_resp <= sp2_small_max_nb();
}

bool use_persistent(sp2_handle_t h) {
  if (h->opt.engine != SP2_ENGINE_TCGEN05 || h->opt.persistent == 2) return false;
  return h->opt.persistent == 1 || h->cur_npad <= kPersistMaxNpad;
}

// enqueue layer launches [first, first + count) on `s`
// pw: the density-only power phase (args_pw, its own work lists)
sp2_status_t enqueue_layers(sp2_handle_t h, int first, int count, cudaStream_t s, int* launches, bool pw = false) {
  const Sp2LayerArgs* A = pw ? h->args_pw : h->args;
  if (use_small(h)) {
    if (count <= 0) return SP2_OK;
    cudaError_t e = sp2_launch_small(A[0], h->cur_npad, s);
    if (e != cudaSuccess) { h->last_cuda_error = (int)e; return SP2_ERR_CUDA; }
    ++*launches;
    return SP2_OK;
  }
  if (use_persistent(h)) {       // the kernel loops until the device controller stops (it starts at layer ctrl->n)
    if (count <= 0) return SP2_OK;
    cudaError_t e = sp2_launch_layers_persistent(h->d_args() + (pw ? 2 : 0), h->cur_cg, pw ? h->n_active_pw : h->n_active, s);
    if (e != cudaSuccess) { h->last_cuda_error = (int)e; return SP2_ERR_CUDA; }
    ++*launches;
    return SP2_OK;
  }
  for (int n = first; n < first + count; ++n) {
    cudaError_t e = sp2_launch_layer(A[n & 1], h->opt.engine, h->cur_cg, s);
    if (e != cudaSuccess) { h->last_cuda_error = (int)e; return SP2_ERR_CUDA; }
    ++*launches;
  }
  return SP2_OK;
}

sp2_status_t enqueue_finalise(sp2_handle_t h, const void* H, sp2_dtype_t in_dt, long ldh, int N, const Pert& P, void* D,
                              sp2_dtype_t out_dt, long ldd, int ring_idx, cudaStream_t s, int* launches,
                              bool refine_only = false) {
  for (int b = 0; b < (P.nb > 0 ? P.nb : 1) && !refine_only; ++b) {   // D (+ D1_0), then D1_b alone for the rest of a batch
    const int zh = P.nb ? 2 + 2 * b : 0, zm = P.nb ? 3 + 2 * b : 1;
    __half* planes[8] = {h->plane(0, 0), h->plane(1, 0), h->plane(0, 1), h->plane(1, 1),
                         h->plane(zh, 0), h->plane(zm, 0), h->plane(zh, 1), h->plane(zm, 1)};
    sp2_launch_finalise(h->ctrl(), planes, h->cur_npad, H, in_dt, ldh, b == 0 ? D : nullptr, P.nb ? P.D1[b] : nullptr, out_dt,
                        ldd, N, b, h->fslots(), s);
    ++*launches;
  }
  if (!refine_only) {
    sp2_launch_finalise_reduce(h->ctrl(), N, h->fslots(), h->ring() + ring_idx, s);
    ++*launches;
  }
  const int nref = h->opt.refine_layers;
  if (nref > 0) {   // float64 refinement layers on the converged iterate; overwrites D, tr D, tr(DH)
    __half* yp[4] = {h->plane(0, 0), h->plane(1, 0), h->plane(0, 1), h->plane(1, 1)};
    CUtensorMap maps[2];                          // the two float64 iterates as TMA tensors (sp2_refine.cu)
    for (int w = 0; w < 2; ++w) {
      int bk = 0, br = 0;
      sp2_refine_box(&bk, &br);
      cuuint64_t gdim[2] = {(cuuint64_t)h->cur_npad, (cuuint64_t)h->cur_npad};
      cuuint64_t gstride[1] = {(cuuint64_t)h->cur_npad * sizeof(double)};
      cuuint32_t box[2] = {(cuuint32_t)bk, (cuuint32_t)br};
      cuuint32_t estr[2] = {1, 1};
      CUresult r = h->encode(&maps[w], CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, h->refine_x(w), gdim, gstride, box, estr,
                             CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                             CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
      if (r != CUDA_SUCCESS) { h->last_cuda_error = 100000 + (int)r; return SP2_ERR_CUDA; }
    }
    const int k = sp2_launch_refine(h->ctrl(), yp, h->cur_npad, N, nref, h->refine_x(0), h->refine_x(1), maps, h->refine_slots(),
                                    h->refine_parts(), h->opt.max_ctas,
                                    H, in_dt, ldh, D, out_dt, ldd, h->ring() + ring_idx, s);
    *launches += k;
  }
  return SP2_OK;
}

// rigorous bounds from the trace of a matrix power (sp2_options_t.power_squarings): a density-only phase of squarings
// before the solve; takes precedence over the Lanczos estimate
bool power_active(sp2_handle_t h, int N, int N_occ) {
  const sp2_options_t& o = h->opt;
  return o.power_squarings > 0 && !o.user_bounds && o.forced_layers <= 0 && N >= 2 && N_occ > 0 && N_occ < N;
}

bool lanczos_active(sp2_handle_t h, int N, int N_occ) {
  const sp2_options_t& o = h->opt;
  return o.lanczos_steps > 0 && !o.user_bounds && !h->no_lanczos && N > 2 * o.lanczos_steps && N_occ > 0 && N_occ < N &&
         !power_active(h, N, N_occ);
}

int effective_max_layers(const sp2_options_t& o) {
  if (o.forced_layers > 0) return o.forced_layers > 64 ? 64 : o.forced_layers;
  return o.max_layers <= 0 ? 100 : (o.max_layers > 126 ? 126 : o.max_layers);
}

// enqueue one whole solve on `s`; the result struct lands in ring[ring_idx].  Only `n_layers` of the
// max_layers layer launches are enqueued (the caller tops up if the solve turns out unfinished:
// k_finalise_reduce then reports SP2_INTERNAL_INCOMPLETE).
sp2_status_t enqueue_solve(sp2_handle_t h, const void* H, const Pert& P, sp2_dtype_t in_dt, long ldh, int N, int N_occ,
                           double tol, void* D, sp2_dtype_t out_dt, long ldd, int ring_idx, cudaStream_t s,
                           int n_layers, int* launches_out, bool close_if_incomplete = false) {
  const int resp = P.nb;
  sp2_status_t st = prepare(h, N, resp, s);
  if (st != SP2_OK) return st;
  const int npad = h->cur_npad;
  const sp2_options_t& o = h->opt;
  const int max_layers = effective_max_layers(o);
  const int forced = o.forced_layers > 0 ? max_layers : 0;
  int launches = 0;
  Sp2Ctrl* c = h->ctrl();
  {   // what this solve may write (sp2_debug_layout)
    const bool trivial = (N_occ == 0 || N_occ == N);
    const size_t nbb = (size_t)sp2_bounds_blocks(N);
    h->touch(h->L.r_ctrl, sizeof(Sp2Ctrl));
    h->touch(h->L.r_ring, (size_t)(ring_idx + 1) * sizeof(sp2_result_t));
    h->touch(h->L.r_bslots, (resp ? h->L.bslots_count + (size_t)resp * nbb : nbb) * sizeof(Sp2BoundSlot));
    if (o.lanczos_steps > 0) h->touch(h->L.r_lanczos, 3 * (size_t)N * sizeof(double));
    if (!trivial) {
      const size_t s_resc = (size_t)sp2_rescale_blocks(npad);
      size_t s_layer = (size_t)sp2_layer_slots(npad, h->cur_cg * h->n_clusters, resp, o.engine);
      h->touch(h->L.r_slots, (s_layer > s_resc ? s_layer : s_resc) * sizeof(Sp2Slot));
      if (resp) h->touch(h->L.r_slots2, (size_t)resp * s_resc * sizeof(Sp2Slot));
      h->touch(h->L.r_fslots, 3 * (size_t)(resp > 1 ? resp : 1) * (size_t)sp2_finalise_blocks(N) * sizeof(double));
      for (int w = 0; w < 2 + 2 * resp; ++w) { h->touch_plane(w, 0, (size_t)npad); h->touch_plane(w, 1, (size_t)npad); }
      if (o.refine_layers > 0 && h->L.r_refine0 >= 0) {
        h->touch(h->L.r_refine0, (size_t)npad * npad * sizeof(double));
        h->touch(h->L.r_refine0 + 1, (size_t)npad * npad * sizeof(double));
        h->touch(h->L.r_refine_slots, refine_slot_doubles((size_t)npad) * sizeof(double));
        h->touch(h->L.r_refine_parts, sp2_refine_parts_bytes(sp2_refine_grid(npad, o.max_ctas)));
      }
    }
  }
  const bool power = power_active(h, N, N_occ);
  if (use_small(h) && !lanczos_active(h, N, N_occ) && !power && N_occ > 0 && N_occ < N) {
    // the smallest problems: prologue, layer stack and finalise in ONE launch of one CTA (sp2_small.cu)
    Sp2SmallProblem sp;
    memset(&sp, 0, sizeof(sp));
    sp.H = H; sp.D = D; sp.ldh = ldh; sp.ldd = ldd;
    for (int b = 0; b < resp; ++b) { sp.H1[b] = P.H1[b]; sp.D1[b] = P.D1[b]; }
    sp.N = N; sp.n_occ = N_occ; sp.max_layers = max_layers; sp.user_bounds = o.user_bounds;
    sp.eps_min = o.eps_min; sp.eps_max = o.eps_max; sp.tol = tol; sp.forced_signs = o.forced_signs;
    sp.forced_layers = forced; sp.no_recentre = o.no_recentre;
    sp.in_f64 = in_dt == SP2_F64; sp.out_f64 = out_dt == SP2_F64; sp.ring_entry = h->ring() + ring_idx;
    if (h->time_layers) SP2_CUDA(h, cudaEventRecord(h->evl0, s));
    SP2_CUDA(h, sp2_launch_small_solve(h->args[0], npad, sp, s));
    ++launches;
    if (h->time_layers) SP2_CUDA(h, cudaEventRecord(h->evl1, s));
    enqueue_finalise(h, H, in_dt, ldh, N, P, D, out_dt, ldd, ring_idx, s, &launches, true);   // float64 refinement, if asked for
    h->launches += (unsigned long long)launches;
    if (launches_out) *launches_out = launches;
    return SP2_OK;
  }
  sp2_launch_init(c, N, N_occ, npad, resp, max_layers, o.user_bounds, o.eps_min, o.eps_max, tol, forced, o.forced_signs, o.no_recentre,
                  power ? o.power_squarings : 0, s);
  ++launches;
  sp2_launch_bounds(H, in_dt, ldh, N, 0, h->bslots(0), s); ++launches;
  for (int b = 0; b < resp; ++b) {    // one slot array of sp2_bounds_blocks(N) per perturbation, contiguous (k_setup)
    sp2_launch_bounds(P.H1[b], in_dt, ldh, N, 1, h->bslots(1) + (size_t)b * sp2_bounds_blocks(N), s);
    ++launches;
  }
  // Lanczos bounds are an estimate (include/sp2.h): skipped for matrices no larger than the Krylov space asked for
  // and on the re-run after the device guard rejected them (SP2_ERR_BOUNDS)
  if (lanczos_active(h, N, N_occ)) {
    sp2_launch_lanczos(c, H, in_dt, ldh, N, o.lanczos_steps, h->lanczos_vecs(), s);
    launches += 2 + 2 * o.lanczos_steps;
  }
  if (power) {
    // power phase: A = (mu I - H)/r0 into the Y planes, power_squarings density-only layers Yhat <- gamma Yhat^2 on the
    // same tensor kernel, then k_power_finish turns ||A^(2^s)||_F into an enclosing interval and hands it to the
    // regular solve below as (device-side) user bounds
    sp2_launch_setup(c, h->bslots(0), sp2_bounds_blocks(N), h->bslots(1), resp ? sp2_bounds_blocks(N) : 0, s); ++launches;
    sp2_launch_rescale(H, in_dt, ldh, c, 0, h->plane(0, 0), h->plane(1, 0), npad, h->slots(), s); ++launches;
    sp2_launch_ctrl0(c, h->slots(), h->slots2(), sp2_rescale_blocks(npad), s); ++launches;
    st = enqueue_layers(h, 0, o.power_squarings, s, &launches, true);
    if (st != SP2_OK) return st;
    sp2_launch_power_finish(c, s); ++launches;
  }
  sp2_launch_setup(c, h->bslots(0), sp2_bounds_blocks(N), h->bslots(1), resp ? sp2_bounds_blocks(N) : 0, s); ++launches;
  if (N_occ == 0 || N_occ == N) {
    sp2_launch_trivial(c, D, resp ? P.D1[0] : nullptr, out_dt, ldd, N, h->ring() + ring_idx, s); ++launches;
    const size_t out_sz = out_dt == SP2_F32 ? 4 : 8;
    for (int b = 1; b < resp; ++b)
      SP2_CUDA(h, cudaMemset2DAsync(P.D1[b], (size_t)ldd * out_sz, 0, (size_t)N * out_sz, N, s));
  } else {
    for (int b = 0; b < resp; ++b) {
      sp2_launch_rescale(P.H1[b], in_dt, ldh, c, 1 + b, h->plane(2 + 2 * b, 0), h->plane(3 + 2 * b, 0), npad,
                         h->slots2() + (size_t)b * sp2_rescale_blocks(npad), s);
      ++launches;
    }
    sp2_launch_rescale(H, in_dt, ldh, c, 0, h->plane(0, 0), h->plane(1, 0), npad, h->slots(), s); ++launches;
    sp2_launch_ctrl0(c, h->slots(), h->slots2(), sp2_rescale_blocks(npad), s); ++launches;
    if (h->time_layers) SP2_CUDA(h, cudaEventRecord(h->evl0, s));
    st = enqueue_layers(h, 0, n_layers, s, &launches);
    if (st != SP2_OK) return st;
    if (h->time_layers) SP2_CUDA(h, cudaEventRecord(h->evl1, s));
    // no top-up is possible without a host round trip (sequence call): an unfinished stack is closed as
    // "not converged, launch budget exhausted" and D is written from the iterate reached
    if (close_if_incomplete && n_layers < max_layers) { sp2_launch_close(c, s); ++launches; }
    enqueue_finalise(h, H, in_dt, ldh, N, P, D, out_dt, ldd, ring_idx, s, &launches);
  }
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) { h->last_cuda_error = (int)e; return SP2_ERR_CUDA; }
  h->launches += (unsigned long long)launches;
  if (launches_out) *launches_out = launches;
  return SP2_OK;
}

sp2_status_t blocking_solve(sp2_handle_t h, const void* H, const Pert& P, sp2_dtype_t in_dt, long ldh, int N, int N_occ,
                            double tol, void* D, sp2_dtype_t out_dt, long ldd, sp2_result_t* out, cudaStream_t s,
                            bool host_buffers, double* tr_d1 = nullptr) {
  const int want_resp = P.nb;
  sp2_status_t st = check_args(h, H, P, in_dt, ldh, N, N_occ, D, out_dt, ldd);
  if (st != SP2_OK) return st;
  if (h->seq_active) return SP2_ERR_INVALID_ARG;
  if (host_buffers && P.nb > 1) return SP2_ERR_INVALID_ARG;
  const void* H1 = P.H1[0]; void* D1 = P.D1[0];
  Pert dP = P;                        // device-side pointers of the perturbations
  const void* dH = H; void* dD = D; void* dD1 = D1;
  long dld_in = ldh, dld_out = ldd;
  const size_t in_sz = in_dt == SP2_F32 ? 4 : 8, out_sz = out_dt == SP2_F32 ? 4 : 8;
  // make sure the launch state is ready before the timed region starts
  st = prepare(h, N, want_resp, s);
  if (st != SP2_OK) return st;
  SP2_CUDA(h, cudaEventRecord(h->ev0, s));
  if (host_buffers) {
    if (!(h->flags & SP2_WITH_HOST_STAGING)) return SP2_ERR_WORKSPACE;
    dH = h->staging(0); dD = h->staging(1);
    dld_in = N; dld_out = N;
    h->touch(h->L.r_staging0, (size_t)N * N * in_sz);
    h->touch(h->L.r_staging0 + 1, (size_t)N * N * out_sz);
    if (want_resp) { h->touch(h->L.r_staging0 + 2, (size_t)N * N * in_sz); h->touch(h->L.r_staging0 + 3, (size_t)N * N * out_sz); }
    SP2_CUDA(h, cudaMemcpy2DAsync(h->staging(0), (size_t)N * in_sz, H, (size_t)ldh * in_sz, (size_t)N * in_sz, N,
                                  cudaMemcpyHostToDevice, s));
    if (want_resp) {
      dP.H1[0] = h->staging(2); dP.D1[0] = dD1 = h->staging(3);
      SP2_CUDA(h, cudaMemcpy2DAsync(h->staging(2), (size_t)N * in_sz, H1, (size_t)ldh * in_sz, (size_t)N * in_sz, N,
                                    cudaMemcpyHostToDevice, s));
    }
  }
  int launches = 0;
  const bool layers_timed = !(N_occ == 0 || N_occ == N);
  // The layer count is only known on the device.  Launch as many layers as the previous solve of this
  // shape needed (+ slack) instead of max_layers early-exit launches; if the solve turns out unfinished,
  // top up once with the rest (the answer is the same: the device controller decides when to stop).
  const int max_layers = effective_max_layers(h->opt);
  float layers_ms = 0.f;
  int bounds_fallback = 0;
  for (int attempt = 0; attempt < 2; ++attempt) {
    int n_first = max_layers;
    if (h->opt.forced_layers <= 0 && h->layers_hint > 0 && h->layers_hint < max_layers) n_first = h->layers_hint;
    h->time_layers = 1;
    int l0 = 0;
    st = enqueue_solve(h, dH, dP, in_dt, dld_in, N, N_occ, tol, dD, out_dt, dld_out, 0, s, n_first, &l0);
    launches += l0;
    h->time_layers = 0;
    if (st != SP2_OK) { h->no_lanczos = 0; return st; }
    for (int pass = 0; pass < 2; ++pass) {
      if (host_buffers) {
        SP2_CUDA(h, cudaMemcpy2DAsync(D, (size_t)ldd * out_sz, dD, (size_t)N * out_sz, (size_t)N * out_sz, N,
                                      cudaMemcpyDeviceToHost, s));
        if (want_resp)
          SP2_CUDA(h, cudaMemcpy2DAsync(D1, (size_t)ldd * out_sz, dD1, (size_t)N * out_sz, (size_t)N * out_sz, N,
                                        cudaMemcpyDeviceToHost, s));
      }
      SP2_CUDA(h, cudaMemcpyAsync(h->h_result, h->ring(), sizeof(sp2_result_t), cudaMemcpyDeviceToHost, s));
      if (tr_d1)    // the pinned result ring is idle outside a sequence: entry 1.. carries tr D1_b
        SP2_CUDA(h, cudaMemcpyAsync(h->h_result + 1, h->ctrl()->tr_d1, sizeof(double) * SP2_MAX_BATCH, cudaMemcpyDeviceToHost, s));
      SP2_CUDA(h, cudaEventRecord(h->ev1, s));
      SP2_CUDA(h, cudaStreamSynchronize(s));
      if (layers_timed) {
        float t = 0.f;
        SP2_CUDA(h, cudaEventElapsedTime(&t, h->evl0, h->evl1));
        layers_ms += t;
      }
      if (h->h_result->status != SP2_INTERNAL_INCOMPLETE || pass == 1) break;
      SP2_CUDA(h, cudaEventRecord(h->evl0, s));                   // top-up: the remaining layer launches
      st = enqueue_layers(h, n_first, max_layers - n_first, s, &launches);
      if (st != SP2_OK) { h->no_lanczos = 0; return st; }
      SP2_CUDA(h, cudaEventRecord(h->evl1, s));
      enqueue_finalise(h, dH, in_dt, dld_in, N, dP, dD, out_dt, dld_out, 0, s, &launches);
      h->launches += (unsigned long long)(max_layers - n_first + 1 + (want_resp > 1 ? want_resp : 1));
    }
    // The Lanczos interval is an estimate.  If the device guard saw an eigenvalue of X leave [0, 1] (or the iterate
    // blow up), solve again with the rigorous Gershgorin discs: same answer as lanczos_steps = 0, one extra pass.
    const int stt = h->h_result->status;
    if (attempt == 0 && lanczos_active(h, N, N_occ) && (stt == SP2_ERR_BOUNDS || stt == SP2_ERR_NONFINITE)) {
      h->no_lanczos = 1; bounds_fallback = 1; h->layers_hint = 0;
      continue;
    }
    break;
  }
  h->no_lanczos = 0;
  float ms = 0.f;
  SP2_CUDA(h, cudaEventElapsedTime(&ms, h->ev0, h->ev1));
  sp2_result_t r = *h->h_result;
  if (r.status == SP2_INTERNAL_INCOMPLETE) r.status = SP2_ERR_CUDA;   // cannot happen: the top-up ran max_layers
  if (r.status == SP2_OK && layers_timed) h->layers_hint = r.layers + 6;
  r.gpu_ms = ms;
  r.layers_ms = layers_ms;
  r.kernel_launches = launches;
  r.bounds_fallback = bounds_fallback;
  if (bounds_fallback) h->layers_hint = 0;       // the Gershgorin re-run's layer count says nothing about the next Lanczos solve
  if (out) *out = r;
  if (tr_d1) {
    const bool trivial = (N_occ == 0 || N_occ == N);
    const double* t = reinterpret_cast<const double*>(h->h_result + 1);
    for (int b = 0; b < P.nb; ++b) tr_d1[b] = trivial ? 0.0 : t[b];
  }
  return (sp2_status_t)r.status;
}

}  // namespace

// ================================================================================================
extern "C" {

size_t sp2_workspace_bytes(int n_max, int flags) {
  if (n_max <= 0 || n_max > SP2_MAX_N) return 0;
  return make_layout(n_max, flags).total;
}

sp2_status_t sp2_create(sp2_handle_t* handle, int n_max, int flags, void* d_workspace, size_t bytes) {
  if (!handle || n_max <= 0 || n_max > SP2_MAX_N) return SP2_ERR_INVALID_ARG;
  *handle = nullptr;
  Layout L = make_layout(n_max, flags);
  if (!d_workspace || (reinterpret_cast<uintptr_t>(d_workspace) & 1023) || bytes < L.total) return SP2_ERR_WORKSPACE;
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return SP2_ERR_CUDA;
  cudaDeviceProp prop;
  if (cudaGetDeviceProperties(&prop, dev) != cudaSuccess) return SP2_ERR_CUDA;
  if (prop.major != 10) return SP2_ERR_ARCH;
  sp2_handle_s* h = new (std::nothrow) sp2_handle_s();
  if (!h) return SP2_ERR_INVALID_ARG;
  if (L.nb_max > 0) flags |= SP2_WITH_RESPONSE;
  h->n_max = n_max; h->flags = flags; h->device = dev; h->num_sms = prop.multiProcessorCount; h->nb_max = L.nb_max;
  h->ws = static_cast<uint8_t*>(d_workspace); h->ws_bytes = bytes; h->L = L;
  default_options(&h->opt);
  h->cur_n = -1; h->cur_npad = -1; h->cur_cg = -1; h->cur_resp = -1; h->cur_seg = -1; h->cur_maxctas = -1; h->n_active = 1; h->cur_pw = -1; h->cur_lock = -1; h->n_active_pw = 1; h->n_flags_pw = 0;
  h->last_cuda_error = 0; h->launches = 0; h->seq_active = 0; h->layers_hint = 0; h->no_lanczos = 0;
  void* fn = nullptr;
  cudaDriverEntryPointQueryResult qres;
  cudaError_t e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres);
  if (e != cudaSuccess || qres != cudaDriverEntryPointSuccess || !fn) { delete h; return SP2_ERR_CUDA; }
  h->encode = reinterpret_cast<PFN_cuTensorMapEncodeTiled_v12000>(fn);
  if (sp2_layer_configure() != cudaSuccess || sp2_refine_configure() != cudaSuccess || sp2_small_configure() != cudaSuccess) {
    delete h; return SP2_ERR_CUDA;
  }
  // The layer kernel is persistent and its last-wave units hand partial sums between CTAs, so every CTA(-pair) of a
  // launch must be able to run at once: size the grid by what the device can keep co-resident, fail here (not
  // with a device-side trap later) if the kernel does not fit at all.
  h->max_clusters[0] = 0;
  for (int cg = 1; cg <= 2; ++cg) {
    cudaError_t oe = sp2_layer_max_coresident(cg, h->num_sms, &h->max_clusters[cg]);
    if (oe != cudaSuccess || h->max_clusters[cg] < 1) { h->last_cuda_error = (int)oe; delete h; return SP2_ERR_CUDA; }
  }
  if (cudaEventCreate(&h->ev0) != cudaSuccess || cudaEventCreate(&h->ev1) != cudaSuccess ||
      cudaEventCreate(&h->evl0) != cudaSuccess || cudaEventCreate(&h->evl1) != cudaSuccess ||
      cudaEventCreateWithFlags(&h->seq_ev[0], cudaEventDisableTiming) != cudaSuccess ||
      cudaEventCreateWithFlags(&h->seq_ev[1], cudaEventDisableTiming) != cudaSuccess) { delete h; return SP2_ERR_CUDA; }
  h->time_layers = 0;
  if (cudaMallocHost(reinterpret_cast<void**>(&h->h_result), sizeof(sp2_result_t) * kRingCap) != cudaSuccess) {
    delete h; return SP2_ERR_CUDA;
  }
  *handle = h;
  return SP2_OK;
}

sp2_status_t sp2_destroy(sp2_handle_t h) {
  if (!h) return SP2_ERR_INVALID_ARG;
  cudaEventDestroy(h->ev0);
  cudaEventDestroy(h->ev1);
  cudaEventDestroy(h->evl0);
  cudaEventDestroy(h->evl1);
  cudaEventDestroy(h->seq_ev[0]);
  cudaEventDestroy(h->seq_ev[1]);
  cudaFreeHost(h->h_result);
  delete h;
  return SP2_OK;
}

sp2_status_t sp2_set_options(sp2_handle_t h, const sp2_options_t* opt) {
  if (!h) return SP2_ERR_INVALID_ARG;
  if (!opt) { default_options(&h->opt); h->layers_hint = 0; return SP2_OK; }
  if (opt->engine != SP2_ENGINE_TCGEN05 && opt->engine != SP2_ENGINE_SIMT_DEBUG) return SP2_ERR_INVALID_ARG;
  if (opt->cta_group < 0 || opt->cta_group > 2) return SP2_ERR_INVALID_ARG;
  if (opt->refine_layers < 0 || opt->refine_layers > 4) return SP2_ERR_INVALID_ARG;
  if (opt->lanczos_steps < 0 || opt->lanczos_steps > 32) return SP2_ERR_INVALID_ARG;
  if (opt->lo_bits != 0 && (opt->lo_bits < 6 || opt->lo_bits > 11)) return SP2_ERR_INVALID_ARG;
  if (opt->seg_kb != 0 && opt->seg_kb != 1 && opt->seg_kb != 2 && opt->seg_kb != 4 && opt->seg_kb != 8 &&
      opt->seg_kb != 16 && opt->seg_kb != 32) return SP2_ERR_INVALID_ARG;
  if (opt->user_bounds && !(opt->eps_max > opt->eps_min)) return SP2_ERR_INVALID_ARG;
  if (opt->persistent < 0 || opt->persistent > 2 || opt->max_ctas < 0) return SP2_ERR_INVALID_ARG;
  if (opt->power_squarings < 0 || opt->power_squarings > 6) return SP2_ERR_INVALID_ARG;
  if (opt->lockstep < 0 || opt->lockstep > 2) return SP2_ERR_INVALID_ARG;
  h->opt = *opt;
  h->layers_hint = 0;
  return SP2_OK;
}

sp2_status_t sp2_get_options(sp2_handle_t h, sp2_options_t* opt) {
  if (!h || !opt) return SP2_ERR_INVALID_ARG;
  *opt = h->opt;
  return SP2_OK;
}

sp2_status_t sp2_density(sp2_handle_t h, const void* dH, sp2_dtype_t in_dtype, long ldh, int N, int N_occ, double tol,
                         void* dD, sp2_dtype_t out_dtype, long ldd, sp2_result_t* out, void* stream) {
  return blocking_solve(h, dH, make_pert(nullptr, nullptr), in_dtype, ldh, N, N_occ, tol, dD, out_dtype, ldd, out,
                        static_cast<cudaStream_t>(stream), false);
}

sp2_status_t sp2_response(sp2_handle_t h, const void* dH, const void* dH1, sp2_dtype_t in_dtype, long ld, int N, int N_occ,
                          double tol, void* dD, void* dD1, sp2_dtype_t out_dtype, long ldo, sp2_result_t* out, void* stream) {
  if (!dH1 || !dD1) return SP2_ERR_INVALID_ARG;
  return blocking_solve(h, dH, make_pert(dH1, dD1), in_dtype, ld, N, N_occ, tol, dD, out_dtype, ldo, out,
                        static_cast<cudaStream_t>(stream), false);
}

sp2_status_t sp2_response_batch(sp2_handle_t h, const void* dH, const void* const* dH1, int nb, sp2_dtype_t in_dtype, long ld,
                                int N, int N_occ, double tol, void* dD, void* const* dD1, sp2_dtype_t out_dtype, long ldo,
                                double* tr_d1, sp2_result_t* out, void* stream) {
  if (!dH1 || !dD1 || nb < 1 || nb > SP2_MAX_BATCH) return SP2_ERR_INVALID_ARG;
  Pert P;
  memset(&P, 0, sizeof(P));
  P.nb = nb;
  for (int b = 0; b < nb; ++b) { P.H1[b] = dH1[b]; P.D1[b] = dD1[b]; }
  double tr_local[SP2_MAX_BATCH];
  return blocking_solve(h, dH, P, in_dtype, ld, N, N_occ, tol, dD, out_dtype, ldo, out, static_cast<cudaStream_t>(stream),
                        false, tr_d1 ? tr_d1 : tr_local);
}

sp2_status_t sp2_density_host(sp2_handle_t h, const void* hH, sp2_dtype_t in_dtype, long ldh, int N, int N_occ, double tol,
                              void* hD, sp2_dtype_t out_dtype, long ldd, sp2_result_t* out, void* stream) {
  return blocking_solve(h, hH, make_pert(nullptr, nullptr), in_dtype, ldh, N, N_occ, tol, hD, out_dtype, ldd, out,
                        static_cast<cudaStream_t>(stream), true);
}

sp2_status_t sp2_response_host(sp2_handle_t h, const void* hH, const void* hH1, sp2_dtype_t in_dtype, long ld, int N,
                               int N_occ, double tol, void* hD, void* hD1, sp2_dtype_t out_dtype, long ldo,
                               sp2_result_t* out, void* stream) {
  if (!hH1 || !hD1) return SP2_ERR_INVALID_ARG;
  return blocking_solve(h, hH, make_pert(hH1, hD1), in_dtype, ld, N, N_occ, tol, hD, out_dtype, ldo, out,
                        static_cast<cudaStream_t>(stream), true);
}

sp2_status_t sp2_sequence_begin(sp2_handle_t h, int N, int N_occ, double tol, int n_steps_hint, void* stream) {
  if (!h || N <= 0 || N > h->n_max || N_occ < 0 || N_occ > N) return SP2_ERR_INVALID_ARG;
  if (n_steps_hint > kRingCap) return SP2_ERR_INVALID_ARG;
  if (h->seq_active) return SP2_ERR_INVALID_ARG;
  h->seq_active = 1; h->seq_N = N; h->seq_nocc = N_occ; h->seq_tol = tol; h->seq_steps = 0;
  h->seq_stream = static_cast<cudaStream_t>(stream);
  return prepare(h, N, 0, h->seq_stream);
}

sp2_status_t sp2_sequence_step(sp2_handle_t h, const void* dH_t, sp2_dtype_t in_dtype, long ldh, void* dD_t,
                               sp2_dtype_t out_dtype, long ldd) {
  if (!h || !h->seq_active) return SP2_ERR_INVALID_ARG;
  if (h->seq_steps >= kRingCap) return SP2_ERR_INVALID_ARG;
  const Pert none = make_pert(nullptr, nullptr);
  sp2_status_t st = check_args(h, dH_t, none, in_dtype, ldh, h->seq_N, h->seq_nocc, dD_t, out_dtype, ldd);
  if (st != SP2_OK) return st;
  // Layer launches per step: what the last FINISHED solve of this shape needed, plus slack (consecutive MD-step
  // Hamiltonians differ little), instead of max_layers launches of which most exit at once.  The hint
  // comes from a blocking call before begin, or from this sequence's own earlier steps: each step leaves an event
  // and a copy of its result in pinned memory, polled here WITHOUT waiting.
  const int max_layers = effective_max_layers(h->opt);
  for (int back = 1; back <= 2 && back <= h->seq_steps; ++back) {   // the two youngest steps still own their events
    const int i = h->seq_steps - back;
    if (cudaEventQuery(h->seq_ev[i & 1]) == cudaSuccess) {
      const sp2_result_t& r = h->h_result[i];
      if (r.status == SP2_OK && r.layers > 0) h->layers_hint = r.layers + kSeqSlack;
      break;
    }
  }
  (void)cudaGetLastError();                                         // "not ready" is not an error
  int n_layers = max_layers;
  if (h->opt.forced_layers <= 0 && h->layers_hint > 0 && h->layers_hint < max_layers) n_layers = h->layers_hint;
  st = enqueue_solve(h, dH_t, none, in_dtype, ldh, h->seq_N, h->seq_nocc, h->seq_tol, dD_t, out_dtype, ldd,
                     h->seq_steps, h->seq_stream, n_layers, nullptr, true);
  if (st != SP2_OK) return st;
  SP2_CUDA(h, cudaMemcpyAsync(h->h_result + h->seq_steps, h->ring() + h->seq_steps, sizeof(sp2_result_t),
                              cudaMemcpyDeviceToHost, h->seq_stream));
  SP2_CUDA(h, cudaEventRecord(h->seq_ev[h->seq_steps & 1], h->seq_stream));
  ++h->seq_steps;
  return SP2_OK;
}

sp2_status_t sp2_sequence_end(sp2_handle_t h, sp2_result_t* results, int* n_steps) {
  if (!h || !h->seq_active) return SP2_ERR_INVALID_ARG;
  h->seq_active = 0;
  const int n = h->seq_steps;
  if (n_steps) *n_steps = n;
  if (n > 0)
    SP2_CUDA(h, cudaMemcpyAsync(h->h_result, h->ring(), sizeof(sp2_result_t) * (size_t)n, cudaMemcpyDeviceToHost,
                                h->seq_stream));
  SP2_CUDA(h, cudaStreamSynchronize(h->seq_stream));
  sp2_status_t worst = SP2_OK;
  for (int i = 0; i < n; ++i) {
    if (results) results[i] = h->h_result[i];
    if (h->h_result[i].status != SP2_OK && worst == SP2_OK) worst = (sp2_status_t)h->h_result[i].status;
    if (h->h_result[i].status == SP2_OK && h->h_result[i].layers > 0) h->layers_hint = h->h_result[i].layers + kSeqSlack;
  }
  return worst;
}

sp2_status_t sp2_congruence(sp2_handle_t h, const void* dZ, const void* dX, sp2_dtype_t in_dtype, long ld, int N,
                            int transpose_first, void* dC, sp2_dtype_t out_dtype, long ldc, void* stream) {
  if (!h || !dZ || !dX || !dC || N <= 0 || N > h->n_max || ld < N || ldc < N) return SP2_ERR_INVALID_ARG;
  if ((in_dtype != SP2_F32 && in_dtype != SP2_F64) || (out_dtype != SP2_F32 && out_dtype != SP2_F64)) return SP2_ERR_INVALID_ARG;
  if (!(h->flags & SP2_WITH_RESPONSE)) return SP2_ERR_WORKSPACE;      // needs the second set of planes
  if (h->seq_active) return SP2_ERR_INVALID_ARG;
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  const int npad = pad_n(N);
  const int cg = pick_cta_group(h, npad, 0);
  const int nt = npad / (128 * cg);
  // launch state of the plain-product mode: every tile, grouped like the layer tiles
  h->tiles_host.clear();
  const int G = 8;
  for (int gi = 0; gi < nt; gi += G)
    for (int gj = 0; gj < nt; gj += G)
      for (int tj = gj; tj < gj + G && tj < nt; ++tj)       // column by column inside a group, as build_tiles
        for (int ti = gi; ti < gi + G && ti < nt; ++ti) h->tiles_host.push_back(make_int2(ti, tj));
  int seg = 4;
  while ((npad / 64) % seg) seg >>= 1;
  const int nC = layer_clusters(h, cg);
  int n_slots = 0;
  build_schedule((int)h->tiles_host.size(), 0, (npad / 64) / seg, nC, h->items_host, h->item_begin_host, &h->n_flags, &n_slots);
  h->n_clusters = nC;
  h->cur_n = -1;                                   // the next solve rebuilds its own launch state
  if (h->items_host.size() > h->L.items_cap || h->tiles_host.size() > h->L.tiles_count ||
      (size_t)n_slots * sp2_layer_scratch_slot_bytes(cg) > h->L.scratch_bytes || h->n_flags > 2 * kMaxClusters)
    return SP2_ERR_WORKSPACE;
  h->touch(h->L.r_tiles, h->tiles_host.size() * sizeof(int2));
  h->touch(h->L.r_items, h->items_host.size() * sizeof(Sp2Item));
  h->touch(h->L.r_item_begin, h->item_begin_host.size() * sizeof(int));
  h->touch(h->L.r_flags, kFlagWords * sizeof(unsigned int));
  h->touch(h->L.r_scratch, (size_t)n_slots * sp2_layer_scratch_slot_bytes(cg));
  h->touch(h->L.r_ctrl, sizeof(Sp2Ctrl));
  h->touch(h->L.r_ring, sizeof(sp2_result_t));
  h->touch(h->L.r_bslots, (h->L.bslots_count + (size_t)sp2_bounds_blocks(N)) * sizeof(Sp2BoundSlot));
  for (int w = 0; w < 4; ++w) h->touch_plane(w, 0, (size_t)npad);
  h->touch_plane(2, 1, (size_t)npad); h->touch_plane(3, 1, (size_t)npad);
  SP2_CUDA(h, cudaMemcpyAsync(h->tiles(), h->tiles_host.data(), h->tiles_host.size() * sizeof(int2), cudaMemcpyHostToDevice, s));
  SP2_CUDA(h, cudaMemcpyAsync(h->items(), h->items_host.data(), h->items_host.size() * sizeof(Sp2Item), cudaMemcpyHostToDevice, s));
  SP2_CUDA(h, cudaMemcpyAsync(h->item_begin(), h->item_begin_host.data(), h->item_begin_host.size() * sizeof(int),
                              cudaMemcpyHostToDevice, s));
  SP2_CUDA(h, cudaMemsetAsync(h->split_flags(), 0, kFlagWords * sizeof(unsigned int), s));
  SP2_CUDA(h, cudaStreamSynchronize(s));
  Sp2Ctrl* c = h->ctrl();
  __half *Lh = h->plane(0, 0), *Lm = h->plane(1, 0), *Xh = h->plane(2, 0), *Xm = h->plane(3, 0), *Th = h->plane(2, 1),
         *Tm = h->plane(3, 1);
  // exponents, then planes: L = Z^T (C = Z^T X Z) or Z (C = Z X Z^T); X is symmetric
  sp2_launch_init(c, N, 0, npad, 0, 1, 0, 0.0, 0.0, 0.0, 0, 0ull, 0, 0, s);
  sp2_launch_bounds(dZ, in_dtype, ld, N, 1, h->bslots(0), s);
  sp2_launch_bounds(dX, in_dtype, ld, N, 1, h->bslots(1), s);
  sp2_launch_gsetup(c, h->bslots(0), h->bslots(1), sp2_bounds_blocks(N), N, h->ring(), s);
  sp2_launch_split(dZ, in_dtype, ld, N, npad, transpose_first ? 1 : 0, 0, c, Lh, Lm, s);
  sp2_launch_split(dX, in_dtype, ld, N, npad, 0, 1, c, Xh, Xm, s);
  int launches = 6;
  Sp2LayerArgs a;
  memset(&a, 0, sizeof(a));
  a.ctrl = c; a.slots = h->slots(); a.tiles = h->tiles(); a.items = h->items(); a.item_begin = h->item_begin();
  a.scratch = h->scratch(); a.flags = h->split_flags(); a.n_flags = h->n_flags; a.n_clusters = nC;
  a.n = N; a.npad = npad; a.n_tiles = (int)h->tiles_host.size(); a.with_response = 0; a.seg_kb = seg;
  a.lo_bits = 11; a.gemm_mode = 1;
  sp2_status_t st;
  // T = L X^T (= L X): planes out
  if ((st = encode_plane_map(h, &a.tm[0], Lh, npad)) != SP2_OK || (st = encode_plane_map(h, &a.tm[1], Lm, npad)) != SP2_OK ||
      (st = encode_plane_map(h, &a.tm[2], Xh, npad)) != SP2_OK || (st = encode_plane_map(h, &a.tm[3], Xm, npad)) != SP2_OK)
    return st;
  a.out[0] = Th; a.out[1] = Tm; a.out_kind = 0;
  cudaError_t e = sp2_launch_layer(a, SP2_ENGINE_TCGEN05, cg, s);
  if (e != cudaSuccess) { h->last_cuda_error = (int)e; return SP2_ERR_CUDA; }
  sp2_launch_gswap(c, s);
  // C = T L^T: the caller's matrix
  if ((st = encode_plane_map(h, &a.tm[0], Th, npad)) != SP2_OK || (st = encode_plane_map(h, &a.tm[1], Tm, npad)) != SP2_OK ||
      (st = encode_plane_map(h, &a.tm[2], Lh, npad)) != SP2_OK || (st = encode_plane_map(h, &a.tm[3], Lm, npad)) != SP2_OK)
    return st;
  a.out_kind = out_dtype == SP2_F64 ? 2 : 1; a.cout = dC; a.ldc = ldc;
  e = sp2_launch_layer(a, SP2_ENGINE_TCGEN05, cg, s);
  if (e != cudaSuccess) { h->last_cuda_error = (int)e; return SP2_ERR_CUDA; }
  launches += 3;
  h->launches += (unsigned long long)launches;
  SP2_CUDA(h, cudaMemcpyAsync(h->h_result, h->ring(), sizeof(sp2_result_t), cudaMemcpyDeviceToHost, s));
  SP2_CUDA(h, cudaStreamSynchronize(s));
  return (sp2_status_t)h->h_result->status;
}

const char* sp2_status_string(sp2_status_t s) {
  switch (s) {
    case SP2_OK: return "ok";
    case SP2_ERR_INVALID_ARG: return "invalid argument";
    case SP2_ERR_WORKSPACE: return "workspace missing, misaligned or too small";
    case SP2_ERR_CUDA: return "CUDA call failed";
    case SP2_ERR_ARCH: return "device is not sm_100";
    case SP2_ERR_NONFINITE: return "non-finite input or iterate";
    case SP2_ERR_DEGENERATE: return "degenerate spectral bounds (eps_max == eps_min)";
    case SP2_WARN_NOT_CONVERGED: return "not converged within max_layers";
    case SP2_ERR_BOUNDS: return "spectral bounds do not enclose the spectrum";
    case SP2_ERR_TOO_LARGE: return "N exceeds the static scratch of the no-allocation entry point (sp2_noalloc_max_n)";
  }
  return "unknown status";
}

int sp2_last_cuda_error(sp2_handle_t h) { return h ? h->last_cuda_error : 0; }
unsigned long long sp2_launch_count(sp2_handle_t h) { return h ? h->launches : 0ull; }

int sp2_debug_schedule(int n_tiles, int with_response, int segs_per_pass, int n_clusters, int* items8, int capacity,
                       int* item_begin) {
  if (n_tiles <= 0 || segs_per_pass <= 0 || n_clusters <= 0) return -1;
  std::vector<Sp2Item> items;
  std::vector<int> begin;
  int n_flags = 0, n_slots = 0;
  build_schedule(n_tiles, with_response, segs_per_pass, n_clusters, items, begin, &n_flags, &n_slots);
  for (size_t i = 0; i < items.size() && (int)i < capacity; ++i) memcpy(items8 + 8 * i, &items[i], sizeof(Sp2Item));
  if (item_begin) for (int c = 0; c <= n_clusters; ++c) item_begin[c] = begin[c];
  return (int)items.size();
}

int sp2_debug_history(sp2_handle_t h, double* tr_x, double* e, int capacity) {
  if (!h) return -1;
  Sp2Ctrl host_ctrl;
  if (cudaMemcpy(&host_ctrl, h->ctrl(), sizeof(Sp2Ctrl), cudaMemcpyDeviceToHost) != cudaSuccess) return -1;
  int cnt = host_ctrl.n + 1;
  if (cnt > SP2_LAYER_CAP) cnt = SP2_LAYER_CAP;
  for (int i = 0; i < cnt && i < capacity; ++i) {
    if (tr_x) tr_x[i] = host_ctrl.tr_x[i];
    if (e) e[i] = host_ctrl.e[i];
  }
  return cnt;
}

sp2_status_t sp2_debug_plane(sp2_handle_t h, int which, size_t* offset, long* pitch, int* exponent, double* shift) {
  if (!h || which < 0 || which > 7) return SP2_ERR_INVALID_ARG;
  const int prev = which >> 2;      // 4..7: the same planes of the PREVIOUS iterate (other ping-pong buffer)
  which &= 3;
  if (which >= 2 && !(h->flags & SP2_WITH_RESPONSE)) return SP2_ERR_INVALID_ARG;
  Sp2Ctrl host_ctrl;
  if (cudaMemcpy(&host_ctrl, h->ctrl(), sizeof(Sp2Ctrl), cudaMemcpyDeviceToHost) != cudaSuccess) return SP2_ERR_CUDA;
  const int buf = (host_ctrl.n & 1) ^ prev;
  if (offset) *offset = (size_t)(reinterpret_cast<uint8_t*>(h->plane(which, buf)) - h->ws);
  if (pitch) *pitch = host_ctrl.npad;
  if (exponent) *exponent = which < 2 ? host_ctrl.t : host_ctrl.u[0];
  if (shift) *shift = host_ctrl.c;
  return SP2_OK;
}

int sp2_debug_layout(sp2_handle_t h, int index, char* name24, size_t* offset, size_t* reserved, size_t* used) {
  if (!h) return -1;
  const int n = (int)h->L.regions.size();
  if (index < 0 || index >= n) return n;
  const Region& r = h->L.regions[index];
  if (name24) memcpy(name24, r.name, sizeof(r.name));
  if (offset) *offset = r.off;
  if (reserved) *reserved = r.reserved;
  if (used) *used = r.used;
  return n;
}

}  // extern "C"
