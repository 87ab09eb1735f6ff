/* b200sht.h -- C ABI of the B200-native spin spherical harmonic / Wigner transform library.
 *
 * Implements the hot path of arXiv 2311.14670 (Price & McEwen): forward and inverse spin-s spherical harmonic
 * transforms and Wigner (SO(3)) transforms, computed with the paper's Wigner d-function recursion along the
 * harmonic order m (Eq. 25-27; renormalised on the fly, Sec. 3.4) fused with
 * the separable theta-ring contraction (Eq. 30 / Eq. 33; Sec. 4.4).
 * The four maps are the paper's problem statement:
 *     F : B_L(S^2) -> C^{L^2},  F^-1,   W : B_L(SO(3)) -> C^{(4L^3-L)/3},  W^-1.
 *
 * Conventions (all entry points)
 *   - Pointers named `f`, `flm`, `flmn`, `work` are DEVICE pointers owned by the caller.  Inputs are never
 *     modified; outputs are fully overwritten (coefficients outside the support |m| <= l, l >= |spin|, |n| <= l
 *     are written as 0).  The library never frees or keeps caller memory beyond the plan's workspace.
 *   - All work is enqueued on `stream`; no entry point synchronises the device except sht_plan_timings().
 *   - Errors are return codes; nothing throws across the ABI.  sht_status_string() names them.
 *   - Layouts are row-major, last index fastest; complex = interleaved (re, im) doubles.
 *       flm  [L][2L-1]            (l, m+L-1)                              embeds C^{L^2}
 *       MW map   f[L][2L-1]       (theta_t, phi_p), theta_t=(2t+1)pi/(2L-1), phi_p=2 pi p/(2L-1)   (Eq. 37-38)
 *       MWSS map f[L+1][2L]       theta_t = 2 pi t/(2L) (t = 0 and t = L are the poles), phi_p = 2 pi p/(2L)              (Eq. 39-40)
 *       DH map   f[2L][2L-1]      theta_t = (2t+1)pi/(4L), phi_p = 2 pi p/(2L-1)                                          (Eq. 34-35)
 *       GL map   f[L][2L-1]       theta_t = acos(x_t), x_t the roots of the Legendre polynomial P_L (north to south)      (Eq. 45)
 *       HEALPix  f[12 nside^2]    ring-ordered: rings north to south, phi increasing within a ring
 *       SO(3)    f[2N-1][L][2L-1] (gamma_g, beta_b, alpha_a), MW in (beta, alpha), gamma_g = 2 pi g/(2N-1)
 *       flmn [2N-1][L][2L-1]      (n+N-1, l, m+L-1)
 *     With reality = 1 (spin 0 only) maps are arrays of real doubles of the same shape, and the m < 0 half of
 *     flm is ignored on input / filled with (-1)^m conj(f_{l,-m}) on output.
 *   - Accumulation order is not fixed: every output element of the fused kernels is the sum of the partial sums of several
 *     degree / ring tiles, added to global memory with fp64 atomics (RED.ADD.F64 / bulk reduce) in whatever order the tiles
 *     finish.  Two runs of the same call therefore agree to rounding (observed <= 1e-15 relative), not bit for bit.
 *   - Band-limit range: Eq. 27 start values are kept as a windowed double plus a one-byte window counter, which reaches down to
 *     2^-122900.  Plan creation returns SHT_EUNSUPPORTED when the smallest start value of the plan's ring sets falls below that
 *     (MW sampling: L above ~9090; HEALPix with L = 2 nside: far beyond nside = 8192).  Nothing is ever silently dropped.
 *   - dtype: SHT_F64, or SHT_F32 (S^2 plans of any sampling and spin, SO(3) plans; BASELINE config 5; adjoints, precompute, the
 *     theta-stage entry points and ring shards return SHT_EUNSUPPORTED with SHT_F32).  With SHT_F32 every public
 *     array is interleaved floats (complex64 / float32); FFTs and staging run in fp64 on internal copies.  S^2, spin 0: the fused
 *     recursion + contraction kernels compute in fp32 (Eq. 25 in the paper's own form, windows of 2^48).  spin != 0 and SO(3): the fp32
 *     kernels recurse the second index n = 0 only, so the fp64 kernels run between the fp32 arrays (fp32 storage, fp64 arithmetic:
 *     about 1e-7).
 *     Accuracy: max|delta| / max|ref| <= 1e-4 (north_star).
 */
#ifndef B200SHT_H
#define B200SHT_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    SHT_OK = 0,
    SHT_EINVAL = 1,        /* bad argument (L < 1, |spin| >= L, N > L, reality with spin != 0, null pointer ...) */
    SHT_EUNSUPPORTED = 2,  /* valid request this build does not implement (fp32, batch > 1) */
    SHT_EWORKSPACE = 3,    /* workspace missing or too small */
    SHT_ECUDA = 4,         /* a CUDA runtime call failed (cudaGetLastError text via sht_last_error()) */
    SHT_ECUFFT = 5         /* a cuFFT call failed */
} sht_status;

enum { SHT_MW = 0, SHT_HEALPIX = 1, SHT_MWSS = 2, SHT_DH = 3, SHT_GL = 4 };   /* sampling */
enum { SHT_F64 = 0, SHT_F32 = 1 };      /* dtype    */
/* plan options (bit flags of sht_plan_s2_opts); 0 = automatic choices.  Results agree to rounding whatever the options. */
enum {
    SHT_OPT_FOLD_ON  = 1u << 0,   /* spin 0: run the recursion on the northern rings only (north-south fold) ...   */
    SHT_OPT_FOLD_OFF = 1u << 1,   /* ... or on all rings.  Default: folded when the northern half alone fills the GPU (MW: L >= 2048) */
    SHT_OPT_INVSYM   = 1u << 2,   /* MW inverse on the L midpoint rings (2j+1)pi/(2L), which are symmetric about the equator -- spin 0: north-south
                                     fold; spin != 0: ONE pass serves order +m at a ring and -m at its mirror ring instead of two passes
                                      -- then an exact FFT resampling of F_m to the MW rings.  Default from L >= 2048 ...       */
    SHT_OPT_NO_INVSYM = 1u << 7,  /* ... this flag keeps the inverse on the rings of the map, every kernel ring written by its own recursion only
                                     (needed for ring shards; on MWSS / DH / GL / HEALPix it selects two passes for spin != 0)             */
    SHT_OPT_TILE64   = 1u << 3,   /* force 64-ring block tiles in the fused kernels ...                                          */
    SHT_OPT_TILE128  = 1u << 4,   /* ... or 128-ring tiles.  Default: 64 when 128-ring tiles give fewer blocks than the device has SMs */
    SHT_OPT_PRECOMPUTE = 1u << 6, /* the paper's full-precomputation mode (Sec. 4.3): the Wigner d-functions of every
                                     (l, m, ring) are computed once at sht_plan_set_workspace and stored -- O(L^3) workspace (16 L^3 to
                                     24 L^3 bytes on MW) -- and the theta steps become plain weighted sums over the stored table
                                     (HBM-bound).  Pays at L <= 512, where the on-the-fly kernels are bound by the latency of their L
                                     sequential recursion steps.  Single-map fp64 S^2 plans; the folds are off. */
    SHT_OPT_ADJOINT  = 1u << 5,   /* also build what the adjoint entry points need (complex fp64 single-map plans; MW / MWSS plans then
                                     carry the tables of two more ring sets: about twice the workspace) */
    SHT_OPT_GRAPH    = 1u << 9,   /* replay each whole transform as ONE captured CUDA graph (one capture per direction and pair of buffers; an
                                     internal capture stream, so the caller's stream may be the default stream).  Default for L <= 512, where a
                                     transform is a chain of 10-50 short launches and bound by launch overhead ...                          */
    SHT_OPT_NO_GRAPH = 1u << 10,  /* ... this flag launches the kernels one by one.  (Stage timing always does.)                          */
    SHT_OPT_NO_SKIP  = 1u << 11,  /* from L >= 1024 the fused kernels skip the "silent head" of a block tile: near the poles every iterate of a tile
                                     stays below the window top for its first p0 steps (nothing is projected there), so the register state after
                                     those steps is computed once at sht_plan_set_workspace and loaded by every transform (about 140 KB of
                                     workspace per tile).  Same results.  This flag runs every step in every transform.                    */
    SHT_OPT_NO_PAIR  = 1u << 8    /* MW / MWSS: the theta-direction FFTs of the forward upsampling and of the symmetric-ring
                                     inverse carry TWO orders m, m+1 per column by default (their extensions to the theta circle are one even
                                     and one odd function, separated afterwards: half the FFT work); this flag keeps one order
                                     per column */
};
enum { SHT_PEAK_DFMA = 0, SHT_PEAK_DMMA = 1, SHT_PEAK_FFMA = 2, SHT_PEAK_FFMA2 = 3 };   /* sht_peak kinds */

typedef struct sht_plan sht_plan;       /* opaque; host object holding sizes, cuFFT handles and table pointers */
typedef void* sht_stream;               /* a cudaStream_t */

const char* sht_status_string(sht_status s);
const char* sht_last_error(void);       /* text of the last CUDA / cuFFT failure on this thread ("" if none) */

/* ---- plans ------------------------------------------------------------------------------------------------
 * A plan fixes (L, spin, sampling, nside, reality) for S^2 or (L, N) for SO(3).  It owns no device memory:
 * the caller provides one workspace of sht_plan_workspace_bytes() bytes (tables + scratch), which
 * sht_plan_set_workspace() fills with the O(L^2) ring / start-value tables ("optionally precompute some
 * additional internal terms ... O(L^2)"; Eq. 27 start values in mantissa/exponent form).
 * The workspace must be 256-byte aligned (SHT_EINVAL otherwise: operand rows are fetched with bulk TMA copies) and must stay
 * valid and untouched while the plan is used.  One plan = one stream at a time; a plan belongs to the device that was current
 * when it was created.  nside is used for HEALPix only (the band-limit L is independent of it).
 * sht_plan_s2_opts() is the general form (batch and option flags SHT_OPT_*); the library reads no environment variables.
 */
sht_status sht_plan_s2(sht_plan** plan, int L, int spin, int sampling, int nside, int reality, int dtype);
sht_status sht_plan_so3(sht_plan** plan, int L, int N, int dtype);
/* the same with option flags: SHT_OPT_ADJOINT (the Wigner adjoints below), SHT_OPT_GRAPH / SHT_OPT_NO_GRAPH; others are ignored */
sht_status sht_plan_so3_opts(sht_plan** plan, int L, int N, int dtype, unsigned opts);
/* A batch of `batch` S^2 problems with identical (L, spin, sampling, reality) transformed together (BASELINE config 5b):
 * the Wigner-d recursion is run once and shared by all maps, which turns the theta / l contraction of Eq. 30 / 33
 * into a dense GEMM per harmonic order m (the einsum of Sec. 4.3, without storing the d-functions); it
 * runs on the FP64 tensor cores.  Arrays gain a leading [batch] axis: f[batch][L][2L-1], flm[batch][L][2L-1].
 * batch = 1 is sht_plan_s2().  The shared-recursion kernels serve MW fp64 plans; on the other samplings and in fp32 a batch is accepted
 * and transformed map by map through the single-map kernels (same arrays, same results, no shared recursion).  The theta-stage entry
 * points below are single-map only. */
sht_status sht_plan_s2_batch(sht_plan** plan, int L, int spin, int sampling, int nside, int reality, int dtype, int batch);
sht_status sht_plan_s2_opts(sht_plan** plan, int L, int spin, int sampling, int nside, int reality, int dtype, int batch, unsigned opts);
int        sht_plan_batch(const sht_plan* plan);
size_t     sht_plan_workspace_bytes(const sht_plan* plan);
sht_status sht_plan_set_workspace(sht_plan* plan, void* work, size_t work_bytes, sht_stream stream);
sht_status sht_plan_destroy(sht_plan* plan);

/* ---- transforms through a plan (device pointers) -----------------------------------------------------------
 * s2_forward : map f -> flm.  MW: FFT in phi (Eq. 31), extension to the torus and upsampling in theta to 2L
 *              rings (the rings are theta'_u = (2u+1) pi/(4L), u = 0..2L-1, on which the
 *              quadrature of Eq. 41-44 is exact for the band-limit-(2L-2) integrand), then the fused recursion
 *              + theta contraction of Eq. 30.
 *              Domain (MW): the last ring of an MW map lies AT theta = pi, where a spin-s function has the single value
 *              c e^{i s phi} (only the order m = s survives, Eq. 29; SO(3): per n, only m = -n).  The transform uses
 *              exactly that component of the ring: its samples are projected onto e^{i s phi} (F_m(pi) := 0 for m != s) before the
 *              torus extension.  For samples of any spin-s function this changes nothing; for arbitrary arrays (e.g. pixel noise
 *              on the pole ring) it makes the result well defined -- it equals the paper's MW(2L)-grid algorithm applied to the
 *              projected array (the paper's algorithm itself is ring-set dependent on inconsistent pole samples, R21).
 *              MWSS: as MW on the theta circle of 2L samples (both pole rings are projected: theta = 0 keeps m = -s, theta = pi keeps
 *              m = s).  DH / GL: explicit quadrature on the rings of the map, weights Eq. 36 / the Gauss-Legendre weights Eq. 46 stands
 *              for (2/((1-x^2) P_L'(x)^2) times 2 pi/(2L-1); Eq. 46 as printed is not that weight, R22).
 *              HEALPix: ring FFTs with phase shift and periodic extension
 *              (PAPER.md:403-407), weights 4 pi/Npix, Eq. 30.
 * s2_inverse : flm -> map f.  Fused recursion + l contraction of Eq. 33, then ring synthesis Eq. 32 (HEALPix:
 *              aliasing fold of F_m onto m mod nphi).
 * so3_forward / so3_inverse : Eq. 15-18: FFT in gamma and one spin -n transform per
 *              n = -(N-1)..N-1, all n batched in the same kernel launches.
 */
sht_status s2_forward_plan(sht_plan* plan, const void* f, void* flm, sht_stream stream);
sht_status s2_inverse_plan(sht_plan* plan, const void* flm, void* f, sht_stream stream);
/* HEALPix forward transform with `niter` refinement iterations (HEALPix has no sampling theorem, "iterations are
 * usually performed"): flm_0 = F f, flm_{k+1} = flm_k + F (f - F^-1 flm_k).  niter = 0 is s2_forward_plan.  HEALPix plans only. */
sht_status s2_forward_iter_plan(sht_plan* plan, const void* f, void* flm, int niter, sht_stream stream);
sht_status so3_forward_plan(sht_plan* plan, const void* f, void* flmn, sht_stream stream);
sht_status so3_inverse_plan(sht_plan* plan, const void* flmn, void* f, sht_stream stream);

/* The hot path alone (the fused recursion + contraction kernels and their pole-ring companions), for timing and
 * for sampled parity at sizes where the full map is too large for the oracle:
 *   s2_theta_inverse_plan: flm -> Fm[2L-1][ntheta] (row m+L-1; ntheta = sht_plan_ntheta(plan, 0)); Eq. 33.
 *   s2_theta_forward_plan: Wm[2L-1][ntheta_q] (row m+L-1; already weighted; ntheta_q = sht_plan_ntheta(plan, 1),
 *                          2L on MW: the rings theta'_u = (2u+1) pi/(4L)) -> flm; Eq. 30.
 */
int        sht_plan_ntheta(const sht_plan* plan, int forward);
sht_status s2_theta_inverse_plan(sht_plan* plan, const void* flm, void* Fm, sht_stream stream);
sht_status s2_theta_forward_plan(sht_plan* plan, const void* Wm, void* flm, sht_stream stream);

/* ---- ring shards: one transform spread over several GPUs ("distributes expensive operations evenly across
 * available devices").  Every ring costs the same number of recursion steps, so the O(L^3) theta step is split by
 * rings: sht_plan_set_shard(plan, rank, nranks) makes the plan serve share `rank` of `nranks` of the rings its fused kernels run
 * on (contiguous shares differing by at most one ring; with the north-south fold a kernel ring stands for a mirror pair).  Arrays
 * keep their full shapes:
 *   forward : the full map in (MW / MWSS: the upsampling mixes rings, so the O(L^2 log L) staging runs in full on every rank; other
 *             samplings read only the shard's rings) -> the PARTIAL flm of the shard's quadrature rings.  The sum over ranks is
 *             the transform: one all-reduce (NCCL, fp64 sum) of L (2L-1) complex numbers.
 *   inverse : the full flm in (replicated) -> a map in which only the shard's rings are filled, all others are zero.  No
 *             collective is needed (each GPU owns its rings); the sum over ranks is the full map.
 * (0, 1) restores the whole transform.  SO(3) plans shard the same way.  SHT_EUNSUPPORTED for batched / fp32 / ADJOINT plans and for
 * MW plans whose inverse runs on the midpoint rings (create the plan with SHT_OPT_NO_INVSYM: the resampling mixes rings).
 * sht_plan_shard_range() reports the share: first kernel ring and count, for the forward or the inverse ring set. */
sht_status sht_plan_set_shard(sht_plan* plan, int rank, int nranks);
sht_status sht_plan_shard_range(const sht_plan* plan, int forward, int* first, int* count);

/* ---- adjoints (Sec. 5.3-5.4): the conjugate transposes of the four maps above, for plans created with
 * SHT_OPT_ADJOINT (SHT_EUNSUPPORTED otherwise).  They are what a vector-Jacobian product of the (linear) transforms needs
 * (VJP = conj(adjoint(conj v)), Eq. 51 / 57).  Same layouts as the transforms; the fused recursion kernels are the existing ones.
 *   s2_forward_adjoint_plan : flm -> map,  F^H.  DH / GL / HEALPix: F^H = Q F^-1 (Eq. 52) -- the inverse transform with every ring
 *                             multiplied by its quadrature weight.  MW / MWSS: the forward transform upsamples, so F^H is the inverse
 *                             theta step ON THE 2L QUADRATURE RINGS, the weights, and the conjugate transposes of the upsampling, the
 *                             torus extension (with the pole-ring projection) and the ring DFT.
 *   s2_inverse_adjoint_plan : map -> flm,  (F^-1)^H = the analysis sum on the rings of the map WITHOUT quadrature weights (Eq. 56;
 *                             F Q^-1 of Eq. 58 where a direct quadrature exists).
 *   s2_theta_forward_adjoint_plan : flm -> Wm[2L-1][ntheta_q], the conjugate transpose of s2_theta_forward_plan (Eq. 62-63 without
 *                             the factor Q_Theta, which that entry point does not apply either).
 *   s2_theta_inverse_adjoint_plan : Fm[2L-1][ntheta] -> flm, the conjugate transpose of s2_theta_inverse_plan (Eq. 67-68).
 * Identities (tests): <F x, y> = <x, F^H y> and <F^-1 c, g> = <c, (F^-1)^H g> to rounding, for arbitrary x, y, c, g.
 */
sht_status s2_forward_adjoint_plan(sht_plan* plan, const void* flm, void* f, sht_stream stream);
sht_status s2_inverse_adjoint_plan(sht_plan* plan, const void* f, void* flm, sht_stream stream);
sht_status s2_theta_forward_adjoint_plan(sht_plan* plan, const void* flm, void* Wm, sht_stream stream);
sht_status s2_theta_inverse_adjoint_plan(sht_plan* plan, const void* Fm, void* flm, sht_stream stream);
/* Wigner transforms (plans from sht_plan_so3_opts with SHT_OPT_ADJOINT): W^H (flmn -> f) and (W^-1)^H (f -> flmn).  Per order n of the
 * gamma transform the Wigner transform is a spin transform with second index n (Eq. 15-18), so its adjoint is the
 * transposed chain: the l-scaling, the S^2 adjoint above for s = -n (one internal S^2 adjoint plan per n, inside the same workspace),
 * the transposed gamma DFT.  Identities (tests): <W x, y> = <x, W^H y>, <W^-1 c, g> = <c, (W^-1)^H g>. */
sht_status so3_forward_adjoint_plan(sht_plan* plan, const void* flmn, void* f, sht_stream stream);
sht_status so3_inverse_adjoint_plan(sht_plan* plan, const void* f, void* flmn, sht_stream stream);

/* Stage timing.  After sht_plan_enable_timing(plan, 1) every transform records CUDA events between its stages;
 * sht_plan_timings() synchronises on the last transform's final event and returns milliseconds:
 *   ms[0] = hot kernels (fused recursion + contraction, incl. pole ring)   -- FP64-pipe bound
 *   ms[1] = FFTs (cuFFT: phi, theta-upsampling, gamma)                     -- HBM bound
 *   ms[2] = staging kernels (transposes, scaling, phases, extension, fold) -- HBM bound
 *   ms[3] = total.
 */
sht_status sht_plan_enable_timing(sht_plan* plan, int on);
sht_status sht_plan_timings(sht_plan* plan, float ms[4]);
/* Algorithmic bytes the last timed transform moved in its FFT (bytes[1]) and staging (bytes[2]) sections: every array a staging
 * kernel, FFT pass or memset reads or writes, counted once (an FFT pass: 32 B per complex element).  bytes[0] (hot) is 0: the
 * fused kernels are compute-bound and are reported in flop (sht_plan_flops).  Divide by sht_plan_timings for GB/s. */
sht_status sht_plan_stage_bytes(const sht_plan* plan, double bytes[3]);

/* ---- the north-star calls: fp64, batch 1, plan + workspace cached inside the library ------------------------
 * (device pointers; the cache allocates its workspaces with cudaMalloc on first use of an argument set and
 * sht_cache_clear() releases them).  HEALPix uses nside = L/2 here (L even).
 * The cache is keyed on (current device, problem).  Calls are thread-safe: an entry is locked while its work is enqueued, and a
 * call on a different stream than the entry's previous call first waits (cudaStreamWaitEvent) for that call's work, so the
 * plan's scratch is never used by two streams at once.  sht_cache_clear() must not race with transforms in flight.
 */
sht_status s2_forward(int L, int spin, int sampling, int reality, const void* f, void* flm, sht_stream stream);
sht_status s2_inverse(int L, int spin, int sampling, int reality, const void* flm, void* f, sht_stream stream);
sht_status so3_forward(int L, int N, const void* f, void* flmn, sht_stream stream);
sht_status so3_inverse(int L, int N, const void* flmn, void* f, sht_stream stream);
sht_status sht_cache_clear(void);

/* ---- host-buffer convenience (end-to-end path): HOST pointers, copies in and out on `stream`, then a stream
 * synchronise.  Same semantics and layouts as above.
 */
sht_status s2_forward_host(int L, int spin, int sampling, int reality, const void* f_host, void* flm_host, sht_stream stream);
sht_status s2_inverse_host(int L, int spin, int sampling, int reality, const void* flm_host, void* f_host, sht_stream stream);
sht_status so3_forward_host(int L, int N, const void* f_host, void* flmn_host, sht_stream stream);
sht_status so3_inverse_host(int L, int N, const void* flmn_host, void* f_host, sht_stream stream);

/* ---- allocation-free entry point -----------------------------------------------------------------------------
 * For callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that forbid it): the theta
 * step of the inverse transform, Eq. 33 with the Wigner d-functions of Eq. 25-29, on caller-given rings -- what
 * s2_theta_inverse_plan computes -- with no plan, no workspace and no cudaMalloc / cudaFree / cuFFT call.  A variant of the stored-table
 * kernels of SHT_OPT_PRECOMPUTE (Sec. 4.3) whose d-function table E[2L-1][ntheta][L] lives in one static device array of
 * SHT_NOALLOC_SCRATCH_BYTES inside the library (every GPU that loads the library holds it until the process exits).
 *   L, spin : band-limit and spin, |spin| < L.
 *   theta   : HOST array of ntheta ring colatitudes in [0, pi] (read before the call returns; pole rings take Eq. 28 / 29).
 *   flm     : DEVICE, complex128 [L][2L-1] (column m + L - 1), read only.
 *   Fm      : DEVICE, complex128 [2L-1][ntheta] (row m + L - 1), every entry written; need not be cleared.
 *   err     : optional HOST buffer of err_len bytes that receives the text of a failure ("" on success); may be NULL.
 * Limits: 1 <= ntheta <= SHT_NOALLOC_MAX_RINGS and (2L-1) * ntheta * L * 8 bytes <= SHT_NOALLOC_SCRATCH_BYTES (e.g. L = 64 on
 * 2L = 128 rings, L = 80 on L rings); beyond them SHT_EUNSUPPORTED with the reason in err, nothing launched.  The two kernels are
 * enqueued on `stream`; the call does not synchronise.  Every call shares the static table (its first kernel rewrites every entry
 * the second reads, so no state carries over between calls): calls that may overlap on the GPU -- different streams without an
 * event between them, or host threads on one device -- race on it and must be ordered by the caller.  fp64, single map. */
#define SHT_NOALLOC_SCRATCH_BYTES (8 << 20)
#define SHT_NOALLOC_MAX_RINGS 128
sht_status s2_theta_inverse_noalloc(int L, int spin, int ntheta, const double* theta, const void* flm, void* Fm, sht_stream stream,
                                    char* err, size_t err_len);

/* ---- measurement helpers: register-only instruction chains, return achieved TFLOP/s and kernel ms (used by bench.py for the
 * roofline denominators, since MEASURED_PEAKS.json has no FP64 / FP32 ALU entries).  kind: SHT_PEAK_DFMA (fma.f64),
 * SHT_PEAK_DMMA (mma.sync.m8n8k4.f64, the FP64 tensor-core path of the batched kernels), SHT_PEAK_FFMA (fma.f32),
 * SHT_PEAK_FFMA2 (packed fma.rn.f32x2, the arithmetic of the fp32 kernels: same peak as FFMA, half the issue slots).
 * sht_fp64_peak() is sht_peak(SHT_PEAK_DFMA, ...). */
sht_status sht_peak(int kind, int iters, double* tflops, float* ms, sht_stream stream);
sht_status sht_fp64_peak(int iters, double* tflops, float* ms, sht_stream stream);

/* ---- introspection --------------------------------------------------------------------------------------- */
/* number of kernels of this library launched by the calling thread since the last reset (bench: gpu_launches) */
long       sht_launch_count(int reset);
/* number of d-steps (one Eq. 25 evaluation for one (l, theta, pass)) one transform of this plan performs */
double     sht_plan_dsteps(const sht_plan* plan, int forward);
/* algorithmic flop of the hot kernels of one transform of this plan: per d-step 6 (Eq. 25 as the paper states it:
 * 1 FMA + 2 MUL + 1 FMA) + 4 per (harmonic order, map) served (Eq. 30 / 33: complex x real multiply-add) */
double     sht_plan_flops(const sht_plan* plan, int forward);
/* share of the block-steps of the fused kernels that a transform of this plan skips (the "silent head" of the block tiles near the poles,
 * SHT_OPT_NO_SKIP; 0 for plans that run every step): those steps project nothing, their effect on the recursion state is loaded from a table */
double     sht_plan_skip_fraction(const sht_plan* plan, int forward);
const char* sht_version(void);

#ifdef __cplusplus
}
#endif
#endif /* B200SHT_H */
