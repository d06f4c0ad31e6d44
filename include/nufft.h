/* nufft.h -- C ABI of the B200-native NUFFT hot path (arxiv 1710.03197, PyNUFFT).
 *
 * What the library computes, stage by stage (citations are PAPER.md lines; readings R1..R20 are listed in
 * DESIGN.md "Readings of the paper"):
 *
 *   forward      A   = V F S         PAPER.md:48-52, eq.(1) :50     scaling :54-56, zero-pad + FFT :58-68,
 *                                                                    interpolation :72-74
 *   adjoint      A^H = S^H F^H V^H   PAPER.md:78-84, eq.(2) :82     gridding :76, IFFT + crop :70
 *   selfadjoint  A^H A               PAPER.md:86-98, eq.(5) :96     applied back to back (R8)
 *   multi-coil   A_multi x = [A(c_i.x)]_i,  A_multi^H y = sum_i conj(c_i).A^H y_i   PAPER.md:251-258, eqs.(34)-(35)
 *   batch mode   several images per call
 *   CG           linear CG on A^H A x = A^H y                       PAPER.md:96, 124-143 (R12)
 *   L1TV-OLS     split Bregman, eqs.(13)-(22)                       PAPER.md:158-198 (R13-R18)
 *
 * Conventions (all binding):
 *   - d in {1,2,3}.  Image x is C-order [batch][N0]([N1]([N2])) complex64; image index n_a sits at position
 *     n_a - N_a/2 (R4).  Samples y are [batch][M] complex64 in the caller's sample order.  om is [M][d] float64,
 *     radians per image sample, axis a of om pairs with image axis a; values outside [-pi,pi) are wrapped.
 *   - forward sign e^{-i om.(n - N/2)}; adjoint is the exact conjugate transpose (no 1/prod(K) factor, R5).
 *   - interpolator: Kaiser-Bessel of width J grid cells ("interpolator size"; J = 6 is the paper's
 *     workload and the tuned path), beta = pi sqrt((J/sigma)^2 (sigma-1/2)^2 - 0.8), sigma = K/N = 2, scaling factors
 *     1/Phi (R1-R3); periodic grid (R7).
 *   - complex64 = two IEEE float32 (re, im), i.e. CUDA float2; declared here as nufft_c64 so that this header
 *     needs no CUDA include.  `stream` arguments are a cudaStream_t passed as void* (NULL = default stream).
 *   - POINTER KINDS.  "host" = ordinary host memory read during the call.  "device" = CUDA device memory,
 *     owned by the caller, 8-byte aligned, valid until the stream work enqueued by the call has finished.
 *     The library never allocates, frees or retains caller arrays, except coil maps (borrowed, see below).
 *   - every call returns 0 (NUFFT_OK) or a negative nufft_status; nothing is printed, nothing throws or aborts.
 *   - transform calls are asynchronous: they enqueue kernels on `stream` and return.  A plan owns one workspace:
 *     use one stream at a time per plan.  Distinct plans are independent.
 *   - a plan belongs to the CUDA device that was current when nufft_plan created it (its buffers and kernel attributes live
 *     there): every later call must be made with that device current, else NUFFT_EINVAL.
 *   - outputs are overwritten, never accumulated into.  In-place (x_in == x_out) is allowed for selfadjoint.
 *   - supported: d in {1,2,3} (1-D: "1D signals"; planar path, atomic V^H only -- adjoint_mode = 1 is
 *     refused); Jd[a] the same on every axis, 2 <= Jd <= 8 (odd widths included);
 *     Kd[a] in {32,64,128,256,512,1024}; Nd[a] even, 2 <= Nd[a] < Kd[a] (the ratio Kd[a]/Nd[a] may differ per axis);
 *     1 <= batch <= max_batch.  Kd == 2 Nd (the paper's and every BASELINE config's ratio) runs the pruned, fused FFT passes;
 *     any other ratio runs the unpruned FFT with S + zero-pad and crop + S^H fused into its contiguous-axis pass, planar layout, and has
 *     no Toeplitz form (nufft_toeplitz_build -> NUFFT_EINVAL); everything else works unchanged.  Jd == 6 runs the tiled / batch-interleaved kernels;
 *     every other width runs the direct V (one thread per sample, prod(J) gathered loads) and, in 2-D, a tiled V^H with the
 *     lane map derived from J (warp-private shared tiles, one TMA reduce-add flush per work item; 1-D / 3-D: one vector
 *     atomic per stencil point into a zeroed grid), planar layout at every batch size, adjoint_mode = 1 refused; all transforms, solvers, density weights and the Toeplitz form work on such plans.
 *     Anything else -> NUFFT_EINVAL (there is no CPU fallback).
 */
#ifndef NUFFT_B200_H
#define NUFFT_B200_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct { float re, im; } nufft_c64;          /* layout-identical to CUDA float2 */
typedef struct nufft_plan_s *nufft_plan_t;

typedef enum {
    NUFFT_OK      =  0,
    NUFFT_EINVAL  = -1,   /* bad d / sizes / Jd / batch / null pointer / unsupported option                 */
    NUFFT_ENOMEM  = -2,   /* host or device allocation failed                                             */
    NUFFT_ECUDA   = -3,   /* a CUDA runtime call failed; nufft_last_cuda_error() gives the cudaError_t    */
    NUFFT_ERANGE  = -4,   /* om contains a non-finite value                                               */
    NUFFT_ESTATE  = -5,   /* call needs something not set (e.g. coil maps)                                */
    NUFFT_ETOOBIG = -6    /* nufft_adjoint_noalloc: prod(Kd) exceeds NUFFT_NOALLOC_MAX_CELLS                 */
} nufft_status;

/* Options.  Zero-initialise or call nufft_default_opts first. */
typedef struct {
    int coef_mode;      /* how V (and the 3-D V^H) get their interpolation weights (north star item 3):
                           0 = recomputed on the fly from a piecewise polynomial fit of the kernel: 4 + 4 d bytes of plan
                               data per sample (the default: fewest bytes; measured 2-7 % slower than 1, profiles/r02_coef_mode.md);
                           1 = precomputed by the plan in float64, rounded once, stored zero-padded in a coalesced per-sample
                               layout in walk order -- 96 B per sample and walk order (48 B in tile order) for the interleaved
                               2-D V, 112 B for the register-window 3-D V / V^H (moved to shared memory by one bulk copy
                               per 16 samples).  Other kernels (planar
                               2-D, generic widths) recompute in either mode; the interleaved V^H always reads its
                               float64-built 96-B table.  Any other value -> NUFFT_EINVAL                                   */
    int adjoint_mode;   /* planar path: 0 = V^H by tile-sorted accumulation on chip, one TMA reduce-add flush per work item
                               (3-D: register windows over pencil-sorted samples, win3d.cuh; 2-D: warp-private shared tiles);
                               summation order across work items free: reproducible to rounding only;
                           1 = deterministic: tiles flushed to private slabs and summed in fixed order
                               (bit-reproducible run to run);
                           2 = 3-D only: the plane-owner shared-memory kernel of round 1 (kept for A/B measurements).
                           The interleaved path (batch >= 12) is always deterministic (gather form, fixed order)        */
    int interp_mode;    /* 0 = library default: register-window kernels -- 3-D planar V keeps an 8 x 8 x 8 window of the
                               staged tile in registers and slides it along the pencil-sorted samples; interleaved V keeps
                               the window (8 x 8, 6 x 10, ... cells) of a group of neighbouring samples in registers; the
                               forward call walks the CALLER's sample order, writing y directly, when the trajectory is
                               coherent (>= 90 % of consecutive samples within two grid cells: radial spokes, spiral arms);
                               A^H A, the solvers and incoherent trajectories walk a tile order whose 19 x 19-cell tiles
                               are staged in shared memory by one tensor-map copy each; 2-D planar V stages tiles likewise;
                           1 = the plain variants: direct gather in 3-D and planar 2-D; on the interleaved path the block-sorted
                               walk with windows loaded from L2 (+ layout pass), never the caller's order or shared tiles;
                           2 = the generic-width kernels (direct V, atomic V^H, planar) even at Jd = 6: what a plan
                               with Jd != 6 runs, selectable at Jd = 6 for cross-checks against the tuned kernels;
                           3 = the round-1 kernels (half-warp-per-sample 3-D V, stencil-per-sample interleaved V), kept
                               for A/B measurements                                                                    */
    int tile[3];        /* tile shape in grid cells per axis, 0 = library default                                */
    int max_subtile;    /* max samples per V^H work item (hot tiles are split), 0 = default                      */
    int use_graphs;     /* 1 = CUDA-graph replay of launch-bound work on a non-default stream (the legacy stream cannot
                               capture: eager launches are used there):
                               - nufft_forward / nufft_adjoint / nufft_selfadjoint: a call whose (batch, pointers, stream)
                                 was seen before is replayed as one graph (small FIFO cache in the plan; the first call of
                                 each kind runs eagerly);
                               - the CG iterations of nufft_solve_cg and of the L1TV solvers' inner solves: one graph per
                                 iteration (pointers are fixed, every scalar lives on the device).  Default 0           */
    int batch_layout;   /* workspace layout of batched 2-D transforms (PAPER.md:52 batch mode, :251-258 coils):
                           0 = auto: calls with batch >= 12 (the measured crossover) use the batch-interleaved grid [group][K0][K1][32]
                               (lanes = images; V^H in gather form with register accumulators, deterministic),
                               smaller batches and 3-D use the planar grid [batch][K0][K1]([K2]);
                           1 = always planar;  2 = interleaved for every batch >= 2 (for measuring the crossover)  */
    int kernel;         /* interpolator ("the default kernel is the min-max kernel [5], other kernel
                               functions can be used"; the paper prints no formula -- DESIGN.md readings R1, R25):
                           0 = Kaiser-Bessel window (reading R1; the library default and the BASELINE configs);
                           1 = min-max interpolator with the Kaiser-Bessel scaling factors: per sample
                               and axis the J REAL weights that minimise the worst-case error over unit-norm images,
                               T w = r(delta) (reading R25).  Same S, F, F^H, S^H and the same kernels: only the weight
                               polynomial (and the float64 V^H table) differ, so every call works unchanged.  The
                               weights depend on N_a: one polynomial per axis                                        */
} nufft_opts;

int nufft_default_opts(nufft_opts *o);

/* Plan creation (everything derived from the trajectory is computed once and offloaded
 * "before iterative algorithms begin").  Nd, Kd: int64[d] host; Jd: int[d] host; om: float64 [M][d] row-major,
 * host, copied (the caller may free it on return).  max_batch >= 1 sizes the workspace grid(s):
 * max_batch * prod(Kd) * 8 bytes of device memory.  opts == NULL selects the defaults.
 * Synchronous (host work + uploads on the default stream).  On failure *out is NULL. */
int nufft_plan(int d, const int64_t *Nd, const int64_t *Kd, const int *Jd,
               int64_t M, const double *om, int max_batch, const nufft_opts *opts, nufft_plan_t *out);

/* y[b][m] = (A x_b)[m], b < batch.   x: device [batch][prod Nd];  y: device [batch][M].   eq.(1) */
int nufft_forward(nufft_plan_t p, int batch, const nufft_c64 *x, nufft_c64 *y, void *stream);

/* x[b] = A^H y_b.   y: device [batch][M];  x: device [batch][prod Nd].   eq.(2) */
int nufft_adjoint(nufft_plan_t p, int batch, const nufft_c64 *y, nufft_c64 *x, void *stream);

/* x_out[b] = A^H A x_in[b], the intermediate samples stay in the plan's workspace.   eq.(5), R8 */
int nufft_selfadjoint(nufft_plan_t p, int batch, const nufft_c64 *x_in, nufft_c64 *x_out, void *stream);

/* x = A^H y for ONE image (eq.(2), the same kernels as nufft_adjoint at batch 1 on the planar path) for callers that
 * cannot tolerate an allocation: code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.
 * The call makes no cudaMalloc / cudaFree and calls no allocating library routine: the oversampled grid that V^H
 * accumulates into and F^H transforms (the scratch of a5 / a4) lives in a file-scope `static __device__` array of the
 * library, NUFFT_NOALLOC_MAX_CELLS complex64 cells = 2 MiB, which every GPU that loads the library holds until the
 * process exits (its device address is taken once per device, at plan creation, with cudaGetSymbolAddress).
 *   y: device [M];  x: device [prod Nd], caller-owned.  Asynchronous on `stream` like nufft_adjoint.
 *   prod(Kd) > NUFFT_NOALLOC_MAX_CELLS -> NUFFT_ETOOBIG (e.g. 512 x 512 and 64^3 grids fit, 1024^2 and 256^3 do not);
 *   plans with adjoint_mode = 1 (their slabs are allocated on first use) and calls made while nufft_profile_enable is
 *   on (events are created) -> NUFFT_EINVAL;  the static array could not be located at plan creation -> NUFFT_ESTATE.
 * The array is SHARED by every plan, stream and thread of the process on that GPU and keeps the last call's contents:
 * the call zero-fills the part it uses before accumulating (the same grid_zero pass as nufft_adjoint), so a call never
 * sees stale data, but two calls that overlap on the GPU (different streams, or different host threads on unordered
 * streams) race on it -- order them on one stream or with events.  The result is that of nufft_adjoint up to the
 * summation order of the tile flushes (adjoint_mode = 0: reproducible to rounding only). */
#define NUFFT_NOALLOC_MAX_CELLS 262144
int nufft_adjoint_noalloc(nufft_plan_t p, const nufft_c64 *y, nufft_c64 *x, void *stream);

/* The same three transforms on HOST buffers (bench.py's end-to-end leg).  x / y are host pointers, read / written
 * asynchronously: they must stay valid until `stream` has passed this call, and should be page-locked (pinned) --
 * pageable memory works but serialises the copies.  The batch is cut into chunks (16 images on the interleaved path: its
 * kernels cost the same for 16 and 32 images, the copies do not, and the pipeline is copy-bound);
 * chunk c+1 is copied in on an internal copy stream while the kernels of chunk c run on `stream` and chunk c-1 is
 * copied back on a second copy stream; `stream` is made to wait for the last copy back before the call's work counts
 * as finished.  Device staging buffers (2 x 2 chunks) belong to the plan.
 * nufft_host_input_ready(p, 1): the caller promises that the host INPUT of every later *_host call is final when the call
 * is made (it is not the target of work still pending on `stream`); the copy in then need not wait for `stream` and may
 * overlap the copy back of the previous call.  Outputs stay stream-ordered.  Default 0 (strict stream order). */
int nufft_host_input_ready(nufft_plan_t p, int on);
int nufft_forward_host(nufft_plan_t p, int batch, const nufft_c64 *x_host, nufft_c64 *y_host, void *stream);
int nufft_adjoint_host(nufft_plan_t p, int batch, const nufft_c64 *y_host, nufft_c64 *x_host, void *stream);
int nufft_selfadjoint_host(nufft_plan_t p, int batch, const nufft_c64 *x_in_host, nufft_c64 *x_out_host, void *stream);

/* The four stages on their own (used by the per-stage parity tests and the per-stage timings).
 * grid: device [batch][prod Kd] complex64 in natural FFT order (k = 0 is index 0), caller-owned.
 *   scale_fft:  grid = F S x          (a1+a2)      fft_scale: x = S^H F^H grid   (a5+a6; grid is DESTROYED)
 *   interp:     y = V grid            (a3)         gridding:  grid = V^H y       (a4; grid fully overwritten) */
int nufft_stage_scale_fft(nufft_plan_t p, int batch, const nufft_c64 *x, nufft_c64 *grid, void *stream);
int nufft_stage_interp   (nufft_plan_t p, int batch, const nufft_c64 *grid, nufft_c64 *y, void *stream);
int nufft_stage_gridding (nufft_plan_t p, int batch, const nufft_c64 *y, nufft_c64 *grid, void *stream);
int nufft_stage_fft_scale(nufft_plan_t p, int batch, nufft_c64 *grid, nufft_c64 *x, void *stream);

/* Multi-coil operator, eqs.(34)-(35) PAPER.md:251-258.  c: device [ncoil][prod Nd], BORROWED: it must stay valid
 * and unchanged until the plan is destroyed or other maps are set.  ncoil <= max_batch.  ncoil = 0 clears.
 *   forward_coils:      y[i] = A (c_i . x)                     x: [prod Nd]   y: [ncoil][M]
 *   adjoint_coils:      x    = sum_i conj(c_i) . A^H y[i]
 *   selfadjoint_coils:  x_out = sum_i conj(c_i) . A^H A (c_i . x_in)                                            */
int nufft_set_coils(nufft_plan_t p, int ncoil, const nufft_c64 *c);
int nufft_forward_coils(nufft_plan_t p, const nufft_c64 *x, nufft_c64 *y, void *stream);
int nufft_adjoint_coils(nufft_plan_t p, const nufft_c64 *y, nufft_c64 *x, void *stream);
int nufft_selfadjoint_coils(nufft_plan_t p, const nufft_c64 *x_in, nufft_c64 *x_out, void *stream);

/* Linear conjugate gradient on the normal equation A^H A x = A^H y, x0 = 0, exactly niter iterations, no
 * preconditioner (eq.(5), :124-143; R12).  If coil maps are set and use_coils != 0 the multi-coil
 * operator is used and y is [ncoil][M]; else y is [M].  x: device [prod Nd] (output).  Scalars (alpha, beta,
 * inner products) are float64 on the device; nothing is read back during the iteration.
 * resnorm_host: NULL, or host double[niter+1] receiving ||r_k||_2, k = 0..niter (forces a stream sync at the end). */
int nufft_solve_cg(nufft_plan_t p, int use_coils, const nufft_c64 *y, nufft_c64 *x, int niter,
                   double *resnorm_host, void *stream);

/* Split-Bregman L1TV-OLS, eqs.(13)-(22) PAPER.md:158-198 with readings R13-R18 (2-D images only):
 *   scale the problem by 1/max|A^H y| (R17); repeat n_outer times { repeat n_inner times { rhs = mu A^H y^k +
 *   lam sum_a grad_a^T(d_a - b_a) (16);  x <- n_cg CG steps on (mu A^H A + lam sum_a grad_a^T grad_a) x = rhs warm
 *   started (15),(17),R16;  d_a = shrink(grad_a x + b_a, 1/lam) (18)-(19);  b_a += grad_a x - d_a (20)-(21) }
 *   A^H y^{k+1} = A^H y^k + A^H y - A^H A x (22) };  result scaled back.
 * grad_a = periodic forward difference along image axis a (eq.(12), R15).
 * y, x as in nufft_solve_cg.  Synchronises the stream once (to read max|A^H y|). */
int nufft_solve_l1tv_ols(nufft_plan_t p, int use_coils, const nufft_c64 *y, nufft_c64 *x,
                         double mu, double lam, int n_outer, int n_inner, int n_cg, void *stream);

/* ---- rows SURVEY.md 8(f) marks "next", built on the same kernels -------------------------------------------------
 * Density compensation, eqs.(6)-(7) PAPER.md:118-122 with reading R21 (w_0 = 1, w real, w <- w / |A A^H w|, exactly
 * niter iterations).  w: device complex64 [M] (output; imaginary parts are 0).
 *   nufft_adjoint_dcf: x[b] = A^H (y_b . w), y device [batch][M], w device [M], x device [batch][prod Nd]. */
int nufft_density_weights(nufft_plan_t p, int niter, nufft_c64 *w, void *stream);
int nufft_adjoint_dcf(nufft_plan_t p, int batch, const nufft_c64 *y, const nufft_c64 *w, nufft_c64 *x, void *stream);

/* Toeplitz form of A^H A ("precomputing A^H A", ref.[6]; reading R22):
 *   A^H A x = crop(F^H(T^ . F(pad x))) on the same K = 2N grid, T^ = F(T), T[d] = sum_m w_m e^{i om_m . d}.
 * nufft_toeplitz_build computes T^ once per plan from 2^d adjoint NUFFTs of the weights w (device complex64 [M], or NULL =
 * all ones), phase-modulated on the host in float64, on the plan's OWN geometry: with d = d' + s, d' in [-N/2, N/2)^d and
 * s in {-N/2, +N/2}^d, T[d' + s] = sum_m (w_m e^{i om_m . s}) e^{i om_m . d'} is the adjoint NUFFT of the modulated weights;
 * every supported size works (no larger grid).  Synchronises the stream.  The result differs from the back-to-back
 * nufft_selfadjoint by the interpolation-kernel error (~1e-5 relative), not by rounding; V and V^H no longer run.
 * nufft_toeplitz_enable(p, 1) makes nufft_solve_cg and the L1TV solvers apply A^H A this way (NUFFT_ESTATE before a build). */
int nufft_toeplitz_build(nufft_plan_t p, const nufft_c64 *w, void *stream);
int nufft_toeplitz_enable(nufft_plan_t p, int on);
int nufft_selfadjoint_toeplitz(nufft_plan_t p, int batch, const nufft_c64 *x_in, nufft_c64 *x_out, void *stream);
int nufft_selfadjoint_toeplitz_coils(nufft_plan_t p, const nufft_c64 *x_in, nufft_c64 *x_out, void *stream);

/* Split-Bregman L1TV-LAD, eqs.(23)-(33) PAPER.md:204-249: L1TV-OLS plus a split of the data term (reading R23: the
 * `b_y^k` printed in eq.(29) is b_f^k; the A^H y of eqs.(29),(32) is the scaled A^H y, not the Bregman-updated one):
 *   rhs = mu (A^H y^k + d_f - b_f) + lam sum_a grad_a^T(d_a - b_a) (25);  x <- n_cg warm-started CG steps on K x = rhs (24),(26);
 *   d_a, b_a as in L1TV-OLS (27)-(28),(30)-(31);  r = A^H A x - A^H y;  d_f = shrink(r + b_f, 1/mu) (29);  b_f += r - d_f (32);
 *   outer: A^H y^{k+1} = A^H y^k + A^H y - A^H A x (33).  Arguments and synchronisation as nufft_solve_l1tv_ols. */
int nufft_solve_l1tv_lad(nufft_plan_t p, int use_coils, const nufft_c64 *y, nufft_c64 *x,
                         double mu, double lam, int n_outer, int n_inner, int n_cg, void *stream);

/* The paper's own conjugate-gradient solution, eqs.(8)-(11) (reading R24): CG on V^H V k = V^H y over the
 * oversampled grid (k_0 = 0, exactly niter iterations, float64 scalars on the device), then x = S^-1 F^-1 k (normalised
 * inverse FFT, crop, divide by the scaling factor; eq.(10)).  y: device [M]; x: device [prod Nd] (output).  Single image,
 * planar path; 5 grid-sized work vectors are allocated on first use.  resnorm_host as in nufft_solve_cg. */
int nufft_solve_cg_kspace(nufft_plan_t p, const nufft_c64 *y, nufft_c64 *x, int niter, double *resnorm_host, void *stream);

/* Plan facts.  Any pointer may be NULL.  bytes_plan = device bytes of per-sample plan data; bytes_work = device
 * bytes of workspace (grids, sample buffers, solver vectors); n_tiles / n_work = V^H tiles and work items (after
 * hot-tile splitting); max_tile_samples = the largest tile's sample count. */
int nufft_plan_info(nufft_plan_t p, int64_t *bytes_plan, int64_t *bytes_work,
                    int64_t *n_tiles, int64_t *n_work, int64_t *max_tile_samples);

/* Modes the plan chose (SURVEY 8(b) "modes chosen").  Any pointer may be NULL.  J = kernel width; kernel = 0
 * Kaiser-Bessel / 1 min-max (opts.kernel); paths = bit mask: 1 = the batch-interleaved 2-D path serves calls with batch >=
 * its threshold, 2 = its V walks the caller's sample order (trajectory-coherent plan), 4 = the generic-width kernels (direct
 * V, atomic V^H) serve the plan, 8 = the Toeplitz operator is enabled; poly_err = max abs error of the degree-9 float32
 * weight polynomial the kernels evaluate against the float64 kernel it was fitted to (weights are <= 1). */
int nufft_plan_modes(nufft_plan_t p, int *J, int *kernel, int *paths, double *poly_err);

/* Tile histogram of the plan (SURVEY 8(b) "tile histogram"): counts[0] = tiles without samples, counts[k] (k >= 1) = tiles
 * holding 2^(k-1) <= n < 2^k samples, k < NUFFT_TILE_HIST_BUCKETS (the last bucket also takes every larger tile).  The tiles
 * are those of the planar V^H / 3-D V kernels (default 16 x 32 cells in 2-D, 8 x 8 x 16 in 3-D); the sum of the
 * counts is n_tiles of nufft_plan_info.  counts: int64[NUFFT_TILE_HIST_BUCKETS], host, written. */
#define NUFFT_TILE_HIST_BUCKETS 24
int nufft_plan_tile_histogram(nufft_plan_t p, int64_t *counts);

/* Number of kernel launches the library has enqueued for this plan since creation (bench.py's gpu_launches). */
int64_t nufft_launch_count(nufft_plan_t p);

/* Per-kernel device timing (bench.py's roofline leg).  While enabled, every kernel the library launches for this
 * plan is bracketed by a pair of CUDA events on the launching stream.  nufft_profile_get synchronises those events
 * and returns, for kernel label i (0 <= i < nufft_profile_count), its name (static string), the summed device time
 * in milliseconds and the number of launches since the last reset.  Timing is off by default (no events recorded). */
int nufft_profile_enable(nufft_plan_t p, int on);
int nufft_profile_reset(nufft_plan_t p);
int nufft_profile_count(nufft_plan_t p);
int nufft_profile_get(nufft_plan_t p, int i, const char **name, double *total_ms, int64_t *launches);

/* Frees the plan, its device buffers, streams, events and cached graphs.  The caller must first synchronise every stream
 * that still has work of this plan enqueued (the library does not wait).  Borrowed coil maps are not freed. */
int nufft_destroy(nufft_plan_t p);

const char *nufft_strerror(int code);
int nufft_last_cuda_error(void);         /* the cudaError_t of the last NUFFT_ECUDA on this thread, else 0 */
const char *nufft_version(void);

#ifdef __cplusplus
}
#endif
#endif /* NUFFT_B200_H */
