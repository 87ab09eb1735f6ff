// internal.h -- shared declarations of the CUDA library (not part of the public ABI; see include/b200sht.h).
//
// Arithmetic scheme of the hot kernels ("e-form"):
//   Eq. 25  d_{m-1} = lambda_m a_{m-1} d_m - (a_{m-1}/a_m) d_{m+1},  a_m = 2/sqrt((l-m)(l+m+1)),
//   is run on e_m = d_m / c_m with c_{m-1} = a_{m-1} kappa_m c_m, c_l = 1, kappa_m = 2^{k_m} a power of two chosen per
//   quantum of SHT_TQ degrees:
//       e_{m-1} = lambda'_m e_m - g'_m e_{m+1},
//       lambda'_m(theta) = lambda_m(theta) s_m,  s_m = 2^{-k_m};     g'_m(l) = (l-m)(l+m+1) G_m,  G_m = 2^{-2-k_m-k_{m+1}}.
//   Both coefficients are separable (theta-only x l-only), so one d-step is 1 DMUL + 1 DFMA.  Everything that depends
//   on (l, m) or (theta, m) alone is an O(L^2) table prepared outside the hot kernels (staging.cu): c_m(l) (folded
//   into the harmonic coefficients on the inverse, into the finalisation on the forward), lambda_m(theta), (s_m, G_m).
//   Renormalisation (Sec. 3.4): the iterate pair carries a power-of-two scale 2^{-480 k}; while
//   k > 0 the stored value stays below 2^-340 (it can grow by at most 2^20 per step between checks), so its
//   (wrong-scale) contribution, even times c_m(l) <= 2^250, is below fp64 resolution and no masking is needed;
//   a check every 8 steps moves the window (k -> k-1) once the stored value exceeds 2^-500.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#define SHT_TWIN (-500)   // window top: stored start values with k > 0 are <= 2^TWIN
#define SHT_SWIN 480      // window stride: true value = stored * 2^(-SWIN*k)
#define SHT_JCHK 8        // steps between window checks
#define SHT_SKIP_STATE_BYTES (64 * 256 * 8 + 9 * 256 * 4)   // per block: 64 doubles + 9 words per compute thread
#define SHT_TQ 64         // quantum of the kappa tables = degrees per block tile of both hot kernels

struct ThetaPass {
    int n;                 // second index of d^l_{m,n} in this pass
    int sgn_out;           // harmonic order served at recursion step m is m_out = sgn_out * m  (P mode)
    int m_end;             // last recursion step (inclusive), <= 0
    int slab;              // which (n-)slab of the in/out arrays this pass belongs to
    int fold;              // forward, n != 0: one pass serves +m from its own ring and -m from the mirrored ring pi - theta via
                           // d^l_{-m,n}(pi - theta) = (-1)^{l-n} d^l_{m,n}(theta); the sign is applied to the -m column
    const double* st_val;  // [Lp][ntp] windowed start values of d^l_{l,n}
    const uint8_t* st_k;   // [Lp][ntp] window counters
    const int* m_lo;       // [ntp] ring theta is served at step m iff m >= m_lo[theta] (nullptr: always)
    const double* lam;     // [m-m_end][ntp] lambda_m(theta) for this pass's second index (plan-time table)
    const double* in;      // inverse: G[m-m_end][Lp][ROWD] rows {c*Re, c*Im (x NC), g'_m(l), s_m}
                           // forward: W[m-m_end][ntp][NC] weighted F_m samples (complex)
    double2* out;          // inverse: F[row][ntp] (row = m_out mod NB)   forward: H[m_out+L-1][Lp]
    const double* pre;     // precompute mode (precompute.cu): E[m-m_end][ntp][Lp] stored e-form d-functions of this pass, else nullptr
};

struct ThetaArgs {
    int L, Lp;             // band-limit, padded (multiple of 128)
    int nth, ntp;          // regular rings, padded (multiple of 128)
    int NB;                // rows of the inverse output (FFT length in phi, 2L-1)
    int ldout;             // inverse: row length of the output F[row][ldout] (= ntp unless the ring set is a folded half)
    int nfull;             // folded ring sets: ring th of the northern half mirrors ring nfull-1-th of the full set
    const double2* sg;     // [Lp/TQ][sgstride] (s_m, G_m) per quantum, column m - mmin
    int sgstride, mmin;
    const double* ctab;    // [m - mmin][Lp] c_m(l) (forward: applied to the reduced sums of each pass)
    const ThetaPass* passes;
    int npass;
    int fold0;             // n = 0, northern rings only (theta_kernels.cu FOLD): forward operand rows hold the E / O sets,
                           // the inverse keeps even-l / odd-l partial sums and writes both rings of a mirror pair
    int th_lo, th_hi;      // ring shard (sht_plan_set_shard): only kernel rings th_lo <= th < th_hi are served by this launch
    int nsm;               // SMs of the device (tile choice)
    // Skipping the silent head of a tile.  For rings near a pole the iterates of a whole tile stay below the
    // window top (every counter k > 0) for the first p0 pairs of steps: nothing is projected there, the recursion merely carries the
    // state.  At plan time the kernels run once in PROBE mode (record, per block, the first pair in which any warp contributed) and once in
    // DUMP mode (run pairs [0, p0) and store the register state); transforms then LOAD that state and start at pair p0.
    int skip_mode;         // 0 = transform (loads the state where skip_p0 > 0), 1 = probe, 2 = dump
    int* skip_p0;          // [block] pairs to skip (multiple of 8), 0 = none; PROBE writes the first contributing pair here
    double* skip_state;    // [block][SHT_SKIP_STATE_BYTES]: e_m, e_{m+1} of the 32 items of the 256 compute threads, window counters, wact
    int tile;              // 0 = automatic, 64 / 128 = forced ring-tile size (plan option SHT_OPT_TILE64 / SHT_OPT_TILE128)
};

// ---- batched path (theta_mma.cu): the contraction of a batch of maps runs on FP64 tensor-core MMAs -----------------
#define SHT_MMA_NCOL 32   // real columns per column group = 16 complex columns (map, +-m)
#define SHT_MMA_ROW 36    // doubles per operand row: 32 columns + 2 side columns + 2 pad (conflict-free LDS.64)
#define SHT_MMA_ROWF 68   // forward rows of the n = 0 fold: 32 columns E + 32 columns O + lambda + 3 pad
// Operand rows, one per (column group, m - m_end, K index), SHT_MMA_ROW doubles:
//   inverse  Gb[cg][m-m_end][Lp][36]:  32 columns c_m(l) scale(l) f_lm (re, im per complex column), [32] g'_m(l), [33] s_m
//   forward  Wb[cg][m-m_end][ntp][36]: 32 columns q(theta) F_m(theta),                                [32] lambda_m(theta)
// Results:   Ob[cg][m-m_end][Mp][32]   (Mp = ntp rings on the inverse, Lp degrees on the forward), accumulated by bulk reduce.
struct MmaArgs {
    int L, Lp, nth, ntp;
    int ncg;                   // column groups (gridDim.z)
    const double2* sg;         // (s_m, G_m) per quantum, as in ThetaArgs
    int sgstride, mmin;
    size_t in_cg_stride, out_cg_stride;   // doubles between column groups of ThetaPass::in / ::out
    int fold0;                 // forward, n = 0: northern rings only, operand rows of SHT_MMA_ROWF doubles (E and O column sets)
    const ThetaPass* passes;   // in = Gb / Wb of the pass, out = Ob of the pass, lam / st_val / st_k / m_lo as in the single-map kernels
    int npass;
};
cudaError_t launch_theta_mma(const MmaArgs& a, bool forward, cudaStream_t st);

// ---- fp32 variant (theta_f32.cu): n = 0, MW sampling, one map ------------------------------------------------------------
struct F32Args {
    int L, Lp, nth, ntp, NB, ldout;
    int fold0;                // northern rings only.  forward: W32 rows hold the E / O sets; inverse: both rings of a mirror pair are written
    int nfull;                // folded ring sets: ring th mirrors ring nfull-1-th
    const float4* ab;         // [m][Lp] {A, A, -B, -B}: A_m(l) = a_{m-1}(l), B_m(l) = a_{m-1}(l)/a_m(l) (Eq. 25-26), duplicated for the packed
                              // two-rings-per-instruction arithmetic; rows m = 0..L-1 (row 0 unused: zeros)
    const float* lam32;       // fp32 copy of the lambda table of the n = 0 pass, row m + 1 (layout of ThetaPass::lam with m_end = 0)
    const float* st_val;      // [Lp][ntp] Eq. 27 start values, windowed: true value = st_val * 2^(-48 st_k)
    const uint16_t* st_k;
    const float2* in;         // inverse: G32[m][Lp][NC] float4 {Re, Re, Im, Im} of scale(l) f_lm; forward: W32[m][ntp/2][NSET][2 NC] float2 =
                              // (ring 2p, ring 2p+1) of q(theta) F_m(theta) (staging.cu k_weight_split_f32)
    double2* out;             // inverse: F[row][ldout]; forward: H[m + L - 1][Lp]   (fp64 accumulators shared with the fp64 staging)
    int skip_mode;            // silent-head skip (see ThetaArgs): 0 = transform, 1 = probe, 2 = dump
    int* skip_p0;             // [block] pairs of steps to skip
    float* skip_state;        // [block][SHT_SKIP_STATE_BYTES_F32]: d_m, d_{m+1} pairs and window counters of the 256 threads
};
#define SHT_SKIP_STATE_BYTES_F32 (80 * 256 * 4)   // per block: 32 + 32 floats + 16 counter words per thread
cudaError_t launch_theta_f32(const F32Args& a, bool forward, int NC, cudaStream_t st);

// launchers (theta_kernels.cu); mode 0 = PM (spin 0 complex: +m and -m from one pass), 1 = P (one order per step)
int theta_tile_rings(const ThetaArgs& a);
cudaError_t launch_theta_inverse(const ThetaArgs& a, int mode, cudaStream_t st);
cudaError_t launch_theta_forward(const ThetaArgs& a, int mode, cudaStream_t st);
// precompute.cu (Sec. 4.3): fill the stored d-function tables of the passes, and the theta steps that read them
cudaError_t launch_pre_fill(const ThetaArgs& a, cudaStream_t st);
cudaError_t launch_pre_inverse(const ThetaArgs& a, int mode, int nrows, cudaStream_t st);
cudaError_t launch_pre_forward(const ThetaArgs& a, int mode, int nrows, cudaStream_t st);
// peaks.cu: register-only instruction chains; kind 0 = DFMA, 1 = DMMA (mma.sync m8n8k4 f64), 2 = FFMA.  Returns flop per launch.
cudaError_t launch_peak(int kind, int iters, int nsm, double* sink, cudaStream_t st, double* flop);
int theta_inverse_rowd(int mode);   // doubles per (m, l) entry of the inverse operand table

void count_launch(int n = 1);
// algorithmic bytes (every array a staging kernel / FFT / memset reads or writes, once) of the work enqueued by the calling thread;
// api.cu attributes them to the open timed section (sht_plan_stage_bytes)
void count_bytes(double bytes);
