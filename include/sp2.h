/* sp2.h -- C ABI of the B200-native (sm_100a) SP2 / DNN-SP2 density-matrix library.
 *
 * What the calls compute (arXiv 2107.02737; PAPER.md = /root/reference/PAPER.md at build time):
 *
 *   D = theta(mu*I - H)                                   PAPER.md:127-135, Eq. 17-18
 *     = the orthogonal projector onto the N_occ lowest eigenvectors of the symmetric,
 *       orthogonalised Hamiltonian H, obtained by the DNN-SP2 recursion
 *       X_0 = (eps_max*I - H)/(eps_max - eps_min),        PAPER.md:145   (input layer W0, B0)
 *       X_{n+1} = X_n^2   or   2 X_n - X_n^2,              PAPER.md:149   (Fig. 1: S_n = S_{n-1}^2 or 2S_{n-1} - S_{n-1}^2)
 *     the branch chosen by trace so that tr X moves toward N_occ, repeated until
 *     the idempotency estimate tr X - tr X^2 stops improving.
 *   D1 = first-order response of D to H -> H + eps*H1, carried through the same layers with the
 *     same branches (BASELINE.json north_star; not printed in the paper, which only names its
 *     consumer):  Z_0 = -H1/(eps_max - eps_min),
 *       Z_{n+1} = X_n Z_n + Z_n X_n   or   2 Z_n - (X_n Z_n + Z_n X_n).
 *   tr(DH) = sum_ij D_ij H_ij with the caller's unscaled H (band energy).
 *
 * Conventions
 *   - Matrices are dense, row-major, symmetric, `ld` = row pitch in ELEMENTS (ld >= N).
 *     Input symmetry: the library uses (H_ij + H_ji)/2, which is H itself when H is exactly symmetric.
 *   - sp2_density / sp2_response / sp2_response_batch / sp2_sequence_* / sp2_congruence: every matrix pointer is a DEVICE pointer owned
 *     by the caller; H, H1 are never written; D, D1 must not alias H, H1 or the workspace.
 *     sp2_density_host / sp2_response_host: every matrix pointer is a HOST pointer (pinned memory
 *     is faster, pageable works); the copies to and from the device are part of the call.
 *   - `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).
 *   - The library allocates NO device memory: the caller passes a device workspace of at least
 *     sp2_workspace_bytes() bytes (e.g. a torch uint8 tensor), 1024-byte aligned, which the handle
 *     uses until sp2_destroy; nothing depends on its initial contents.  One handle = one call in flight (not
 *     re-entrant).  The layer kernels are persistent (one CTA per SM): their last-wave units hand partial sums between
 *     CTAs and, up to N = 2048, all layers of a solve run in one launch with a grid-wide barrier in between, so every
 *     CTA of a launch must be resident at once.  sp2_create sizes the grid by what the device can keep co-resident
 *     (cudaOccupancyMaxActiveClusters) and fails with SP2_ERR_CUDA if the kernel does not fit at all; at run time that
 *     needs the SMs to be free, so run ONE solve per GPU at a time, or leave SMs to other work with
 *     sp2_options_t.max_ctas: two solves on different streams of the same GPU can starve each other's CTAs (a
 *     device-side watchdog then traps, SP2_ERR_CUDA, instead of hanging).  The float64 refinement layers follow the
 *     same rule (one block per SM, at most max_ctas of them; their last tiles are split between blocks).
 *   - Every call returns an sp2_status_t; nothing throws, nothing prints.  The blocking calls
 *     enqueue all kernels on `stream`, synchronise that stream once, and fill *out (a HOST struct).
 *   - There is no CPU fallback: on a device that is not compute capability 10.x the calls return
 *     SP2_ERR_ARCH.
 */
#ifndef SP2_B200_H
#define SP2_B200_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

#if defined(__GNUC__)
#define SP2_API __attribute__((visibility("default")))
#else
#define SP2_API
#endif

typedef struct sp2_handle_s* sp2_handle_t;

typedef enum {
  SP2_OK = 0,
  SP2_ERR_INVALID_ARG = 1,   /* null pointer, N <= 0, N > n_max, N_occ outside [0,N], ld < N, bad dtype */
  SP2_ERR_WORKSPACE = 2,     /* workspace null, misaligned or too small */
  SP2_ERR_CUDA = 3,          /* a CUDA runtime / driver call failed (sp2_last_cuda_error) */
  SP2_ERR_ARCH = 4,          /* device is not sm_100 */
  SP2_ERR_NONFINITE = 5,     /* H (or H1) holds NaN/Inf, or the iterate became non-finite */
  SP2_ERR_DEGENERATE = 6,    /* eps_max == eps_min (H = c*I): no spectral width to rescale */
  SP2_WARN_NOT_CONVERGED = 7, /* max_layers reached, or the parameter-free stop fired away from N_occ (degenerate level at the
                                Fermi energy); D (and D1) are still written */
  SP2_ERR_BOUNDS = 8,        /* an eigenvalue of X left [0,1]: the spectral bounds (user_bounds, or a Lanczos estimate in a
                                sequence step) do not enclose the spectrum of H; detected on the device from
                                tr X - tr X^2 < 0 far from convergence; D is not written.  The blocking calls re-run a
                                solve whose LANCZOS bounds fail this check with Gershgorin discs (result.bounds_fallback) */
  SP2_ERR_TOO_LARGE = 9      /* sp2_density_noalloc only: N exceeds sp2_noalloc_max_n() (the library's static scratch);
                                nothing was launched -- use a handle with a workspace for larger problems */
} sp2_status_t;

typedef enum { SP2_F32 = 0, SP2_F64 = 1 } sp2_dtype_t;

/* flags of sp2_workspace_bytes / sp2_create */
#define SP2_WITH_RESPONSE 1     /* room for the first-order iterate Z (sp2_response) */
#define SP2_WITH_HOST_STAGING 2 /* room for device copies of H, H1, D, D1 (the *_host calls), f64-sized */
#define SP2_WITH_REFINEMENT 4   /* room for two float64 N x N iterates (sp2_options_t.refine_layers > 0) */
#define SP2_MAX_BATCH 8         /* perturbations one sp2_response_batch call can carry */
#define SP2_WITH_BATCH(nb) (((nb) & 15) << 8) /* room for nb first-order iterates (implies SP2_WITH_RESPONSE) */

/* layer engines (sp2_options_t.engine) */
#define SP2_ENGINE_TCGEN05 0 /* product path: TMA + tcgen05.mma + TMEM */
#define SP2_ENGINE_SIMT_DEBUG 1 /* slow FP32-FMA scaffold on the same planes/epilogue; tests only, N <= 4096 */

typedef struct {
  int max_layers;   /* default 100, capped at 126 */
  int user_bounds;  /* 0: Gershgorin discs (default); 1: use eps_min/eps_max below (must enclose the spectrum) */
  double eps_min, eps_max;
  int engine;       /* SP2_ENGINE_* (default SP2_ENGINE_TCGEN05) */
  int forced_layers;      /* debug: > 0 runs exactly this many layers, no stop test */
  unsigned long long forced_signs; /* debug: with forced_layers, bit n = 1 -> layer n is X^2, else 2X - X^2 */
  int cta_group;    /* 0 = auto; 1 = 128x128 tiles, one CTA; 2 = 256x256 tiles on a CTA pair (cta_group::2) */
  int lanczos_steps; /* 0 = off (default: Gershgorin bounds only); 1..32: that many Lanczos steps on H tighten the spectral
                        bounds to [theta_min - beta_k, theta_max + beta_k] where that is inside the Gershgorin interval:
                        fewer layers for dense matrices (the paper leaves accelerated variants aside).
                        This interval is a HEURISTIC, not an enclosure (a start vector orthogonal to an extreme
                        eigenvector never sees it): the device guards every solve (SP2_ERR_BOUNDS) and the blocking calls
                        fall back to Gershgorin discs on their own.  Ignored when N <= 2 * lanczos_steps */
  int refine_layers; /* 0 = off (default); 1..4: float64 SP2 layers applied to the converged iterate before D is written
                        (the paper uses 2); D1 is not refined.  Needs SP2_WITH_REFINEMENT */
  int seg_kb;       /* 0 = default (8 up to N = 8192, 4 up to N = 24576, 2 above); 1, 2, 4, 8, 16 or 32 (must divide
                       npad/64): k-blocks of 64 accumulated inside the tensor core before the FP32 round-to-nearest add in
                       registers (shorter = less truncation bias, more drains) */
  int lo_bits;      /* 0 = default (11: full FP16 lo plane); 6..10: round the lo planes to that many significant bits.
                       The B200 is power-capped during the layer stack and multiplier inputs with fewer toggling bits
                       draw less power: lo_bits = 8 measured 1.8 % faster at ~3x larger max|dD|, still > 1000x inside
                       the bar; kept as an experiment knob, not a recommendation */
  int no_recentre;  /* debug, with forced_layers only: keep c on the scalar map instead of the cluster midpoint */
  int persistent;   /* how the layer stack is launched.  0 = auto: N <= 128 (and at most 2 perturbations): ONE CTA with the
                       iterate resident in shared memory, nothing leaves the SM between layers; N <= 2048: ONE persistent
                       launch of the multi-CTA kernel with a grid-wide barrier between layers; above: one launch per layer.
                       1 = the persistent multi-CTA kernel at any size; 2 = one launch per layer at any size */
  int max_ctas;     /* 0 = one CTA per SM (default); > 0: use at most this many CTAs for the layer kernel, e.g. to leave SMs
                       to other work on the same GPU (the layer grid must be co-resident, see "Conventions") */
  int power_squarings; /* 0 = off (default: Gershgorin bounds only); 1..6: RIGOROUS tighter bounds from the trace of a
                       matrix power.  Before the solve, A = (H - mu I)/r0 (mu = tr H/N) is squared s = power_squarings
                       times on the same tensor kernel (density-only layers); since max_i |lambda_i - mu|^p <= tr (H - mu I)^p
                       for even p, r = ||A^(2^s)||_F^(1/2^s) r0 bounds every eigenvalue's distance from mu, whatever the
                       eigenvectors are (no start vector, unlike lanczos_steps), with r <= N^(1/2^(s+1)) rho.  The solve then
                       uses [mu - r, mu + r] (widened by 1e-3 r, intersected with the Gershgorin discs).  Costs s density
                       layers, saves ~2 log2(Gershgorin width / 2r) layers; takes precedence over lanczos_steps */
  int lockstep;     /* launch-per-layer mode (N > 2048): 0 = auto (on from N = 7168), 1 = on, 2 = off.  On: the TMA producer
                       of a CTA checks in every 16 k-blocks and runs ahead only when 7/8 of the grid's producers have
                       reached the same point, so CTAs that stream the same panels stay coincident in L2 (a third
                       fewer DRAM reads per layer at N = 8192, a third of them left at N = 16384).  A hint only: a
                       producer that waits longer than about half a work item free-runs for the rest of the launch,
                       so sharing the device with other streams costs the saving, not progress.  Results are bitwise
                       the same either way. */
} sp2_options_t;

typedef struct {
  int status;                        /* sp2_status_t of the solve */
  int layers;                        /* number of layers applied (paper: 14-16 for water) */
  unsigned long long sign_mask[2];   /* bit n = 1 if layer n was X^2 ('+'), 0 if 2X - X^2 ('-') */
  int stop_reason;                   /* 1 tol, 2 floor (parameter-free), 3 idempotent on entry, 4 max_layers, 5 trivial N_occ, 6 forced,
                                        7 a sequence step ran out of enqueued layer launches (status NOT_CONVERGED) */
  int reserved;                      /* number of float64 refinement layers applied */
  double tr_d;                       /* tr D (should be N_occ) */
  double tr_dh;                      /* sum_ij D_ij H_ij */
  double tr_d1;                      /* tr D1 (should be 0); 0 when no response */
  double idem_est;                   /* last idempotency estimate e_L = tr X_L - tr X_L^2 */
  double eps_min, eps_max;           /* spectral bounds used by the input layer */
  float gpu_ms;                      /* device time of the call (CUDA events on `stream`), blocking calls only */
  float layers_ms;                   /* device time of the layer-kernel launches alone (a3-a5), blocking calls only */
  int kernel_launches;               /* kernels of this library launched by the call */
  int bounds_fallback;               /* 1: the Lanczos bounds failed the device guard and the solve was re-run with Gershgorin discs */
} sp2_result_t;

/* Largest supported dimension (the largest size the GPU parity tests cover; 32-bit index arithmetic in the
 * kernels holds up to here). */
#define SP2_MAX_N 32768

/* Bytes of device workspace needed for problems up to n_max (flags: SP2_WITH_*). 0 if n_max <= 0 or > SP2_MAX_N. */
SP2_API size_t sp2_workspace_bytes(int n_max, int flags);

/* Create a handle on the CURRENT device over caller-owned device memory. */
SP2_API sp2_status_t sp2_create(sp2_handle_t* handle, int n_max, int flags, void* d_workspace, size_t bytes);
SP2_API sp2_status_t sp2_destroy(sp2_handle_t handle);

/* NULL restores the defaults. */
SP2_API sp2_status_t sp2_set_options(sp2_handle_t handle, const sp2_options_t* opt);
SP2_API sp2_status_t sp2_get_options(sp2_handle_t handle, sp2_options_t* opt);

/* H (N x N, in_dtype, pitch ldh) -> D (N x N, out_dtype, pitch ldd).  tol > 0: stop as soon as
 * 0 <= tr X - tr X^2 <= tol with |tr X - N_occ| < 0.5; tol <= 0: parameter-free stop only.
 * N_occ = 0 -> D = 0; N_occ = N -> D = I.  Blocking (one stream synchronise). */
SP2_API sp2_status_t sp2_density(sp2_handle_t handle, const void* dH, sp2_dtype_t in_dtype, long ldh,
                         int N, int N_occ, double tol,
                         void* dD, sp2_dtype_t out_dtype, long ldd,
                         sp2_result_t* out, void* stream);

/* As sp2_density, plus H1 -> D1 (same dtypes and pitches as H / D).  Needs SP2_WITH_RESPONSE. */
SP2_API sp2_status_t sp2_response(sp2_handle_t handle, const void* dH, const void* dH1, sp2_dtype_t in_dtype, long ld,
                          int N, int N_occ, double tol,
                          void* dD, void* dD1, sp2_dtype_t out_dtype, long ldo,
                          sp2_result_t* out, void* stream);

/* Batched response ("preconditioned Krylov subspace approximation" of the kernel
 * needs the response of the same H to several perturbations per MD step): nb perturbations H1_b ride ONE stack
 * of layers, Y^2 is formed once per layer and Y Z_b + Z_b Y once per perturbation, every Z_b with its own plane
 * exponent.  dH1 / dD1 are HOST arrays of nb DEVICE pointers (same dtype and pitch as H / D); tr_d1 is a HOST
 * array of nb doubles (may be NULL) that receives tr D1_b (out->tr_d1 = tr D1_0).  1 <= nb <= the nb given to
 * SP2_WITH_BATCH at create (1 with plain SP2_WITH_RESPONSE).  Blocking.  No host-buffer twin. */
SP2_API sp2_status_t sp2_response_batch(sp2_handle_t handle, const void* dH, const void* const* dH1, int nb,
                                sp2_dtype_t in_dtype, long ld, int N, int N_occ, double tol,
                                void* dD, void* const* dD1, sp2_dtype_t out_dtype, long ldo,
                                double* tr_d1, sp2_result_t* out, void* stream);

/* Host-buffer twins: hH/hH1/hD/hD1 are HOST pointers; H2D and D2H copies run on `stream` inside the
 * call.  Need SP2_WITH_HOST_STAGING (and SP2_WITH_RESPONSE for the response twin). */
SP2_API sp2_status_t sp2_density_host(sp2_handle_t handle, const void* hH, sp2_dtype_t in_dtype, long ldh,
                              int N, int N_occ, double tol,
                              void* hD, sp2_dtype_t out_dtype, long ldd,
                              sp2_result_t* out, void* stream);
SP2_API sp2_status_t sp2_response_host(sp2_handle_t handle, const void* hH, const void* hH1, sp2_dtype_t in_dtype, long ld,
                               int N, int N_occ, double tol,
                               void* hD, void* hD1, sp2_dtype_t out_dtype, long ldo,
                               sp2_result_t* out, void* stream);

/* Consecutive MD-step Hamiltonians (one density-matrix construction per time step).
 * begin fixes N, N_occ, tol and the stream; each step enqueues one density solve and returns
 * without synchronising (per-step results land in a device ring of n_steps_hint entries, at most
 * 4096); end synchronises once and copies the results of the steps issued since begin. */
SP2_API sp2_status_t sp2_sequence_begin(sp2_handle_t handle, int N, int N_occ, double tol, int n_steps_hint, void* stream);
SP2_API sp2_status_t sp2_sequence_step(sp2_handle_t handle, const void* dH_t, sp2_dtype_t in_dtype, long ldh,
                               void* dD_t, sp2_dtype_t out_dtype, long ldd);
SP2_API sp2_status_t sp2_sequence_end(sp2_handle_t handle, sp2_result_t* results, int* n_steps);

/* Congruence transform of a symmetric matrix X with a (general) matrix Z, the step either side of the solver in a
 * non-orthogonal basis (H_orth = Z^T H Z, D = Z D_orth Z^T with Z^T S Z = I):
 *   transpose_first = 1:  C = Z^T X Z        transpose_first = 0:  C = Z X Z^T
 * Device pointers, row-major, pitch ld (Z, X) / ldc (C); X symmetric.  Two products on the same tcgen05 mainloop as the
 * layers (FP16 hi/lo planes, FP32 accumulation in k-segments, ~22-bit operands).  Needs SP2_WITH_RESPONSE (it borrows the
 * second set of planes).  Blocking; C must not alias Z, X or the workspace. */
SP2_API sp2_status_t sp2_congruence(sp2_handle_t handle, const void* dZ, const void* dX, sp2_dtype_t in_dtype, long ld, int N,
                                    int transpose_first, void* dC, sp2_dtype_t out_dtype, long ldc, void* stream);

/* Diagnostics. */
/* ---- no-allocation entry point ------------------------------------------------------------------------------------
 * sp2_density_noalloc: the density matrix of a SMALL problem (2 <= N <= sp2_noalloc_max_n() = 128, 0 < N_occ < N) without
 * a handle, a workspace or any allocation: for callers that cannot call cudaMalloc (code under CUDA graph capture,
 * tight serving loops, harnesses that forbid it).  Same operation as sp2_density with default options (Gershgorin
 * rescale, SP2 layers with the trace rule and the parameter-free stop): ONE launch of the one-CTA
 * kernel that keeps the iterate in shared memory.  The global scratch that kernel needs (final hi/lo planes of both
 * ping-pong buffers, control block, result entry: sp2_noalloc_scratch_bytes() = 134 912 bytes, 132 KB) is a file-scope
 * `static __device__` array inside the library, which every GPU that loads the library holds until the process exits.
 *   dH, dD      device pointers, row-major, pitches ldh / ldd >= N in elements, dtypes as given; owned by the caller
 *   d_result    optional DEVICE pointer: the kernel writes the result struct there (else into the static scratch)
 *   out         optional HOST pointer: if non-NULL the call copies the result struct back and synchronises `stream`
 *               before it returns (return value = out->status); if NULL the call only enqueues (returns SP2_OK when
 *               the launch was accepted; the solve's status is in *d_result once the stream reaches that point)
 *   stream      cudaStream_t, NULL = default stream; the device is the calling thread's current device
 * Errors: SP2_ERR_TOO_LARGE for N > sp2_noalloc_max_n() (nothing launched), SP2_ERR_INVALID_ARG (null pointer, N < 2,
 * N_occ outside (0, N), pitch < N, bad dtype, tol < 0), SP2_ERR_ARCH off sm_100, SP2_ERR_CUDA, and the solve's own
 * statuses.  Calls no cudaMalloc / cudaFree / allocating library routine.  The first call on each device does a
 * one-time set-up (cudaFuncSetAttribute, cudaGetSymbolAddress): make it outside stream capture.
 * EVERY call on a device shares the one scratch array, which keeps the last call's contents (the kernel overwrites all
 * of it and needs none of it zeroed): calls that overlap on the GPU (two streams, two host threads) RACE on the
 * control block and the result entry -- serialise them on one stream, or use handles. */
SP2_API sp2_status_t sp2_density_noalloc(const void* dH, sp2_dtype_t in_dtype, long ldh, int N, int N_occ, double tol,
                                         void* dD, sp2_dtype_t out_dtype, long ldd, sp2_result_t* d_result,
                                         sp2_result_t* out, void* stream);
SP2_API int sp2_noalloc_max_n(void);             /* 128 */
SP2_API size_t sp2_noalloc_scratch_bytes(void);  /* bytes of static device memory per GPU */

SP2_API const char* sp2_status_string(sp2_status_t status);
SP2_API int sp2_last_cuda_error(sp2_handle_t handle);            /* cudaError_t of the last failing CUDA call, 0 if none */
SP2_API unsigned long long sp2_launch_count(sp2_handle_t handle); /* kernels launched through this handle so far */

/* Test hooks (used by tests/ only; stable but not part of the paper's problem statement).
 * Per-layer trace history of the last solve: tr X_n and e_n = tr X_n - tr X_n^2, n = 0..layers. Returns count. */
SP2_API int sp2_debug_history(sp2_handle_t handle, double* tr_x, double* e, int capacity);
/* Byte offset inside the workspace, pitch (elements) and power-of-two exponent of an internal
 * 16-bit plane after the last solve: which = 0 Y.hi, 1 Y.lo, 2 Z.hi, 3 Z.lo of the FINAL iterate
 * (X_L = c*I + (hi+lo)*2^-exp); which + 4 = the same plane of the previous iterate X_{L-1} (other
 * ping-pong buffer; exponent and shift are still those of X_L).  c is returned in *shift. */
SP2_API sp2_status_t sp2_debug_plane(sp2_handle_t handle, int which, size_t* offset, long* pitch, int* exponent, double* shift);

/* The carved regions of the workspace and how much of each the calls made through this handle so far were entitled
 * to write (computed from the launch geometry, not from the allocation formulas).  index in [0, count): fills name24
 * (24 bytes, NUL-terminated), byte offset inside the workspace, reserved bytes, used bytes; any pointer may be NULL.
 * Returns the number of regions (also for an out-of-range index, e.g. -1).  tests/test_gpu_canary.py fills the
 * workspace with a sentinel and checks that used <= reserved and that nothing outside [offset, offset + used) changed:
 * the stand-in for compute-sanitizer, which is not available on the GPU pool. */
SP2_API int sp2_debug_layout(sp2_handle_t handle, int index, char* name24, size_t* offset, size_t* reserved, size_t* used);

/* Host-only: the static work lists of the layer kernel for n_tiles upper-triangular tiles,
 * segs_per_pass k-segments per product pass and n_clusters CTA(-pair)s.  Each item is 8 ints
 * {unit, seg0, seg1, kind (0 whole, 1 contributor, 2 owner), slot, nparts, flag_id, 0}; item_begin has
 * n_clusters + 1 entries.  Returns the number of items (-1 on bad arguments). */
SP2_API int sp2_debug_schedule(int n_tiles, int with_response, int segs_per_pass, int n_clusters, int* items8,
                               int capacity, int* item_begin);

#ifdef __cplusplus
}
#endif
#endif /* SP2_B200_H */
