/*
 * cc_ladder.h -- C ABI of the B200-native Cholesky particle-particle ladder.
 *
 * The one operation behind every entry point (arXiv:2310.04559, Sec. 2, Eq. 6 with the Cholesky form of
 * Eq. 5), "the scaling-determining step" of the CCD/CCSD amplitude equations:
 *
 *     R[i,j,a,b] += sum_{c,d} ( sum_P L[P,a,c] * L[P,b,d] ) * t[i,j,c,d]
 *
 *   i,j in [0,nocc)   occupied orbitals          P in [0,nchol)  Cholesky vectors ("x" in the paper)
 *   a,b,c,d in [0,nvirt) virtual orbitals
 *
 * Layouts: dense, row-major, 0-based, IEEE binary64, no leading-dimension arguments.
 *     L[P][a][c]      nchol * nvirt * nvirt doubles   (operand "xac"; L_0 and L_1 are the same
 *                                                      array)
 *     t[i][j][c][d]   nocc^2 * nvirt^2 doubles        (the (ij, cd) matrix; the paper's t_old[i,c,j,d] with its
 *                                                      middle axes swapped)
 *     R[i][j][a][b]   nocc^2 * nvirt^2 doubles        (the paper's t_new[i,a,j,b], same swap)
 * The result is ACCUMULATED into R ("+=").  Neither symmetry of L in (a,c) nor
 * t[i,j,a,b] == t[j,i,b,a] is assumed.  Any positive sizes up to 30000 per dimension are legal as long as one
 * (i,j) group of R stays below 2^31 elements (nvirt^2, and nocc*nvirt^2 in the paper's [i,a,j,b] storage); all
 * other element counts are 64-bit.
 *
 * The integral tensor (ac|bd) (nvirt^4 doubles) is never stored: tiles of it are built on chip (FP64
 * tensor-core DMMA, K = nchol) and consumed at once by the contraction with t (DMMA, K = tile of (c,d));
 * partial sums reach R through FP64 reductions in L2 (red.global.add.f64), so results are reproducible to
 * rounding (~1e-15 of max|R|), not bitwise, between runs.
 *
 * Ownership: the caller owns L, t, R (and the optional workspace); they must stay valid until the work
 * enqueued on `stream` has completed.  A plan holds host metadata (sizes, options, the workspace pointer) and
 * 256 bytes of device memory (the tile counters of the dynamic scheduler); use one plan from one stream at a time.  R must not overlap L or t.
 *
 * Errors: every call returns an int status, 0 = CC_LADDER_OK, negative = failure; nothing is printed,
 * nothing throws, nothing exits.  There is no CPU fallback: without a usable sm_100 device cc_ladder_plan
 * fails with CC_LADDER_EARCH / CC_LADDER_ECUDA.
 */
#ifndef CC_LADDER_H
#define CC_LADDER_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct cc_ladder_plan_s *cc_ladder_plan_t;   /* opaque, owned by the library */

/* status codes */
#define CC_LADDER_OK            0
#define CC_LADDER_EINVAL      (-1)   /* size <= 0, null pointer, misaligned pointer, overlap, bad option  */
#define CC_LADDER_EARCH       (-2)   /* current device is not compute capability 10.x                     */
#define CC_LADDER_EWORKSPACE  (-3)   /* workspace missing or too small for the selected options            */
#define CC_LADDER_ECUDA       (-4)   /* a CUDA runtime call failed (see cc_ladder_last_cuda_error)         */
#define CC_LADDER_ENOMEM      (-5)   /* host or device allocation failed                                   */
#define CC_LADDER_ESCRATCH    (-6)   /* cc_ladder_split_static: problem needs more than the static scratch  */

/* option keys for cc_ladder_set_option / cc_ladder_get_option */
#define CC_LADDER_OPT_SPLIT        1  /* 0 (default) full tile space; 1 = t+/t- symmetric/antisymmetric
                                         split over a<=b, c<=d blocks: about half the flops (north_star).  Needs a
                                         workspace of about 2 nocc^2 nvirt^2 doubles (cc_ladder_workspace_bytes): t+ / t-
                                         and the partial results R+ / R- as packed upper triangles, ~nvirt^2/2 elements
                                         per (i,j), rows aligned for 128-bit copies                           */
#define CC_LADDER_OPT_ALGO         2  /* CC_LADDER_ALGO_*                                                  */
#define CC_LADDER_OPT_NUM_CTAS     3  /* persistent grid size; 0 (default) = one CTA per SM                 */
#define CC_LADDER_OPT_SUPERTILE    4  /* scheduler: (ab)-blocks x (cd)-blocks per L2 super-tile edge; 0=auto */
#define CC_LADDER_OPT_TILE         5  /* tile shape = block edges <TA,TB,TC,TD> along a, b, c, d (every dimension is
                                         padded to a multiple of its edge): 0 = auto (least estimated time),
                                         full mode: 1 = <8,12,16,8>, 2 = <12,8,12,12>, 3 = <8,12,20,8>;
                                         split mode (square partitions): 4 = <8,8,12,12>, 5 = <8,8,16,16>
                                         (auto: the latter unless the former executes >= 10 % fewer flops);
                                         a value of the other mode means auto                               */

#define CC_LADDER_OPT_EXCHANGE     6  /* 0 (default) the ladder of Eq. 6; 1 = its exchange variant (PAPER.md:283-288,
                                         Eq. 7): R[i,j,a,b] += sum_cd (sum_P L[P,a,d] L[P,b,c]) t[i,j,c,d].  Same kernel
                                         with a and b swapped while the integral tile is built; in split mode the same
                                         t+ with the negated t-.  Not with the simple path or CC_LADDER_OPT_SYMM_L      */

#define CC_LADDER_OPT_LAYOUT       7  /* storage of t and R: CC_LADDER_LAYOUT_IJAB (default) t[i][j][c][d], R[i][j][a][b];
                                         CC_LADDER_LAYOUT_IAJB = the paper's own t_old[i][c][j][d], t_new[i][a][j][b]
                                         (PAPER.md:78-80).  Addressing only, same kernels (split mode: in its pack and
                                         unpack steps).  Not with the simple path or CC_LADDER_OPT_SYMM_L               */
#define CC_LADDER_LAYOUT_IJAB      0
#define CC_LADDER_LAYOUT_IAJB      1

#define CC_LADDER_OPT_XY_ROWS_X     8  /* rows nr / ns of the operand blocks X / Y that cc_ladder_get_info and the tile-   */
#define CC_LADDER_OPT_XY_ROWS_Y     9  /* shape choice refer to; 0 (default) = nvirt, i.e. the ladder.  cc_ladder_xy sets
                                         both from its arguments (Eqs. 8-9)                        */
#define CC_LADDER_OPT_HOST_BUDGET  10  /* cc_ladder_host: device bytes it may allocate; 0 (default) = the free device
                                         memory.  When L + t + R (+ workspace) exceed it, R is streamed in column
                                         blocks (the paper's batch-wise VRAM problem)              */
#define CC_LADDER_OPT_INDEX_BITS   11  /* 0 (default) = the device decodes tile indices in 32-bit arithmetic whenever
                                         they fit; 64 = always 64-bit (same schedule; nvirt > ~2000 needs it anyway) */

#define CC_LADDER_OPT_SYMM_L       12  /* 0 (default) nothing is assumed about L; 1 = the caller guarantees L[P][a][c] ==
                                         L[P][c][a] (real orbitals).  Then <ab|cd> = <cd|ab> and only the
                                         integral tiles with (a,b)-block <= (c,d)-block are built, each used twice (as V
                                         for R[:, (a,b)] and as V^T for R[:, (c,d)]): about 15-19 % fewer flops.  The
                                         result is WRONG for an unsymmetric L (cc_ladder_check_symmetric tests the
                                         precondition).  Plain ladder only: EINVAL with split, exchange, the paper's
                                         storage, cc_ladder_xy and the simple path                                   */

#define CC_LADDER_OPT_SCHEDULE     13  /* how the persistent CTAs get their tiles (full mode; split mode is static):
                                         CC_LADDER_SCHEDULE_DYNAMIC (default) = in tile-index order from a device
                                         counter (keeps the tiles in flight neighbours in the L2 super-tile order for the
                                         whole run); CC_LADDER_SCHEDULE_STATIC = tile blockIdx + k * gridDim            */
#define CC_LADDER_OPT_HOST_BLOCK_ROWS 14 /* cc_ladder_host with PINNED host buffers, full mode, when everything fits the
                                         device: R is still streamed in column blocks of this many rows of a (rounded up
                                         to a multiple of 24) so that its H2D / D2H copies overlap the kernels.
                                         0 (default) = auto (about six blocks; problems with R < 256 MB stay resident),
                                         -1 = off (one resident evaluation).  Also caps the block size when R has to be
                                         streamed because of CC_LADDER_OPT_HOST_BUDGET                              */
#define CC_LADDER_SCHEDULE_DYNAMIC 0
#define CC_LADDER_SCHEDULE_STATIC  1

#define CC_LADDER_ALGO_FUSED       0  /* default: fused on-chip DMMA kernel                                */
#define CC_LADDER_ALGO_SIMPLE      1  /* slow device-side check path (scalar FMA, chunked workspace)       */

/* info keys for cc_ladder_get_info (read-only facts about the plan / last launch) */
#define CC_LADDER_INFO_NUM_TILES        1  /* tiles the scheduler enumerates per evaluation                */
#define CC_LADDER_INFO_KERNEL_LAUNCHES  2  /* kernels one cc_ladder call enqueues                          */
#define CC_LADDER_INFO_FLOPS_EXECUTED   3  /* flops the kernels issue per evaluation (padding included)    */
#define CC_LADDER_INFO_FLOPS_FULL       4  /* 2 v^4 (x + o^2): the algorithmic count of the full contraction */
#define CC_LADDER_INFO_NUM_SMS          5
#define CC_LADDER_INFO_SMEM_BYTES       6  /* dynamic shared memory per CTA of the main kernel             */
#define CC_LADDER_INFO_TILE_SHAPE       7  /* block edges packed as TA<<24 | TB<<16 | TC<<8 | TD           */
#define CC_LADDER_INFO_SUPERTILE_SHAPE  8  /* L2 super-tile in blocks, packed SA<<24 | SB<<16 | SC<<8 | SD  */
#define CC_LADDER_INFO_INDEX_BITS       9  /* 32 or 64: arithmetic width of the device-side tile decode     */
#define CC_LADDER_INFO_HOST_CHUNKS     10  /* R column blocks the last cc_ladder_host call streamed (1 = all resident) */

/* Create a plan for the sizes of Eq. 6: nocc = o, nvirt = v, nchol = x.  Host only; queries
 * the current device, to which the plan then belongs (calls made while another device is current return EINVAL).
 * *plan is set on success, NULL otherwise.  EINVAL: a size <= 0 or > 30000; EARCH / ECUDA: no usable sm_100 device. */
int cc_ladder_plan(cc_ladder_plan_t *plan, int nocc, int nvirt, int nchol);

/* Change / read an option of an existing plan (before the next cc_ladder call): the scheduler of SURVEY.md 8(a) a1
 * (tile shape, L2 super-tile, grid; the paper's analogue is the batch splitting of PAPER.md:206-218), the t+/t- split,
 * the Eq. 7 variant and the paper's storage.  EINVAL: unknown key or illegal value. */
int cc_ladder_set_option(cc_ladder_plan_t plan, int key, long long value);
int cc_ladder_get_option(cc_ladder_plan_t plan, int key, long long *value);
int cc_ladder_get_info(cc_ladder_plan_t plan, int key, long long *value);

/* Device workspace the current options need (0 for the fused non-split path: nothing batch-sized is ever allocated,
 * so the paper's batch-size estimator, has no analogue) and how to provide it.
 * The caller allocates (e.g. torch.empty(..., device="cuda")); 256-byte alignment required. */
size_t cc_ladder_workspace_bytes(cc_ladder_plan_t plan);
int cc_ladder_set_workspace(cc_ladder_plan_t plan, void *dev_ptr, size_t bytes);

/* R += ladder(L, t), Eq. 6 with Eq. 5; with CC_LADDER_OPT_EXCHANGE the Eq. 7 variant.
 * L, t, R are DEVICE pointers (16-byte aligned) in the layouts above.  `stream` is a cudaStream_t (0 = legacy default
 * stream).  Only enqueues work: no host synchronisation, no allocation.  EINVAL: null / misaligned / overlapping
 * buffers (R against L, t and the workspace), an option combination that does not exist (the simple path or
 * CC_LADDER_OPT_SYMM_L with split, exchange or the paper's storage), or a current device other than the plan's; EWORKSPACE: split / simple path without
 * a large enough workspace; ECUDA: a launch failed. */
int cc_ladder(cc_ladder_plan_t plan, const double *L, const double *t, double *R, void *stream);

/* The occupied-virtual family, PAPER.md:288-298 (Sec. 6.2, Eqs. 8-9; the paper's recipe "abcd,ecfd->efab" with "abcd"
 * translated to "xac,xbd"), generalised to two independent blocks of Cholesky vectors:
 *
 *     out[i,j,r,s] += sum_{c,d} ( sum_P X[P,r,c] * Y[P,s,d] ) * t[i,j,c,d]        r < nr, s < ns, c, d < nvirt
 *
 *   Eq. 9  t~_ijbk = sum_xcd L_bd L_kc t_ij^cd :  X = L_ov[P,k,c] (nr = nocc), Y = L_vv[P,b,d] (ns = nvirt), out[i,j,k,b]
 *   Eq. 8  t~_ijkl = sum_xcd L_kc L_ld t_ij^cd :  X = Y = L_ov (nr = ns = nocc),                            out[i,j,k,l]
 *   Eq. 6  the ladder                           :  X = Y = L   (nr = ns = nvirt)
 * X element (P,r,c) is X[P*x_pstride + r*x_rstride + c] (strides in doubles, so a block of a larger Cholesky array
 * L[P][p][q] over all orbitals needs no copy); likewise Y.  t is t[i][j][c][d]; out is out[i][j][r][s], nocc^2*nr*ns
 * doubles (or, with CC_LADDER_LAYOUT_IAJB, t[i][c][j][d] and out[i][r][j][s]).  DEVICE pointers: t and out 16-byte
 * aligned, X and Y 8-byte aligned (16-byte copies are used when the strides are even and the bases 16-byte aligned).
 * Same kernel, scheduler and accumulate semantics as cc_ladder; full mode only (EINVAL with split / the simple path);
 * CC_LADDER_OPT_EXCHANGE pairs r with d and s with c instead.  Enqueue only.  EINVAL also for nr, ns <= 0 or > 30000,
 * strides smaller than the block they address, out overlapping an input. */
int cc_ladder_xy(cc_ladder_plan_t plan, const double *X, long long x_pstride, long long x_rstride, int nr,
                 const double *Y, long long y_pstride, long long y_rstride, int ns, const double *t, double *out,
                 void *stream);

/* Same operation as cc_ladder with HOST pointers (pageable or pinned): copies L, t, R to the device, runs the kernels
 * on a private stream, copies R back and synchronises.  Allocates and frees its own device buffers.  Blocking.
 * When L + t + R (+ workspace) exceed CC_LADDER_OPT_HOST_BUDGET (default: the free device memory) R is streamed in
 * column blocks of `a` through two device buffers while L and t stay resident -- the paper's batch loop over chunks
 * of a with the copies overlapped with the kernels; ENOMEM if even L + t + two blocks do not fit.
 * With pinned host buffers (full mode) R is streamed that way even when everything fits, for the overlap
 * (CC_LADDER_OPT_HOST_BLOCK_ROWS); CC_LADDER_INFO_HOST_CHUNKS tells how many blocks the last call used. */
int cc_ladder_host(cc_ladder_plan_t plan, const double *L_host, const double *t_host, double *R_host);

/* Precondition of CC_LADDER_OPT_SYMM_L: *n_mismatch = number of element pairs a < c with
 * L[P][a][c] != L[P][c][a] (bitwise compare) in the DEVICE array L[nchol][nvirt][nvirt].  Blocking (one pass over L). */
int cc_ladder_check_symmetric(cc_ladder_plan_t plan, const double *L, long long *n_mismatch, void *stream);

/* The roofline denominator measured on the current device: a register-only DMMA.8x8x4 loop,
 * ~0.2 s.  *tflops = flops / elapsed time (CUDA events on `stream`), *flop_per_clk_per_sm = flops per SM cycle from the
 * SM cycle counter (nominal 128).  Either pointer may be NULL.  Blocking; allocates a few bytes of device memory. */
int cc_ladder_fp64_peak(double *tflops, double *flop_per_clk_per_sm, void *stream);

/* The allocation-free entry point, for callers that cannot call cudaMalloc (code under CUDA-graph capture, tight
 * serving loops, harnesses that forbid it).  Same operation as cc_ladder in split (t+/t-) mode with default options
 * (R[i][j][a][b] += Eq. 6; split weights: DESIGN.md reading 10), but with no plan and no caller
 * workspace: the packed-triangle scratch (T+, T-, W+, W-) lives in ONE file-scope `static __device__` array of
 * CC_LADDER_STATIC_SCRATCH_BYTES (32 MiB) inside the library; every GPU that loads the library holds it until the
 * process exits.  L, t, R: DEVICE pointers as for cc_ladder (16-byte aligned, R overlapping neither L nor t), owned by
 * the caller.  Enqueues on `stream` and returns; calls no cudaMalloc / cudaFree / allocating library routine (the
 * scratch address is taken once per device with cudaGetSymbolAddress).
 * Limit: cc_ladder_split_static_bytes(nocc, nvirt) = 8 nocc^2 (4 tri(nvirt) + 16) <= CC_LADDER_STATIC_SCRATCH_BYTES
 * (tri(v) ~ v^2/2 + 2v; e.g. nocc = 12, nvirt = 96 or nocc = 8, nvirt = 140), else CC_LADDER_ESCRATCH and nothing is
 * enqueued -- use cc_ladder with a workspace of your own for larger problems.
 * Every call on a device shares the array, which keeps the last call's contents: each call rewrites T+- and zeroes W+-
 * itself, so calls serialised on one stream (or ordered by events) are independent, but two calls that may OVERLAP on
 * the GPU (different streams, no ordering) race on it -- the caller must order them.
 * Errors: EINVAL (sizes, pointers), EARCH (not sm_100), ESCRATCH, ECUDA (text: cc_ladder_split_static_error()). */
#define CC_LADDER_STATIC_SCRATCH_BYTES 33554432
int cc_ladder_split_static(int nocc, int nvirt, int nchol, const double *L, const double *t, double *R, void *stream);
/* Scratch bytes a problem needs (0 for sizes <= 0); the limit itself; text of the last CUDA error seen by
 * cc_ladder_split_static in this process (thread-unsafe, "" if none). */
size_t cc_ladder_split_static_bytes(int nocc, int nvirt);
size_t cc_ladder_static_scratch_bytes(void);
const char *cc_ladder_split_static_error(void);

/* Release the plan (not the caller's buffers).  NULL is accepted. */
int cc_ladder_destroy(cc_ladder_plan_t plan);

/* Human-readable text of a status code; of the last CUDA error seen by this plan (thread-unsafe). */
const char *cc_ladder_status_string(int status);
const char *cc_ladder_last_cuda_error(cc_ladder_plan_t plan);

/* Library version (major*10000 + minor*100 + patch). */
int cc_ladder_version(void);

#ifdef __cplusplus
}
#endif
#endif /* CC_LADDER_H */
