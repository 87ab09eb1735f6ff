// internal.h -- shared declarations of the CUDA library (not part of the public ABI; see include/b200sht.h).
//
// Arithmetic scheme of the hot kernels ("e-form"; DESIGN.md section "Kernel arithmetic"):
//   Eq. 25  d_{m-1} = lambda_m a_{m-1} d_m - (a_{m-1}/a_m) d_{m+1},  a_m = 2/sqrt((l-m)(l+m+1)),
//   is run on e_m = d_m / c_m with c_{m-1} = a_{m-1} kappa_m c_m, c_l = 1, kappa_m = 2^{k_m} a per-tile power of two:
//       e_{m-1} = lambda'_m e_m - g'_m e_{m+1},
//       lambda'_m(theta) = lambda_m(theta) 2^{-k_m},     g'_m(l) = (l-m)(l+m+1) 2^{-2-k_m-k_{m+1}}.
//   Both coefficients are separable (theta-only x l-only), so one d-step is 1 DMUL + 1 DFMA; the (l,m)-only factor
//   c_m(l) is folded into the harmonic coefficients (inverse) or into the reduced sums (forward).
//   Renormalisation (Sec. 3.4): the iterate pair carries a power-of-two scale 2^{-480 k}; while
//   k > 0 the stored value stays below 2^-340 (it can grow by at most 2^20 per step between checks), so its
//   (wrong-scale) contribution, even times c_m(l) <= 2^280, is below fp64 resolution and no masking is needed;
//   a check every 8 steps moves the window (k -> k-1) once the stored value exceeds 2^-500.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#define SHT_TWIN (-500)   // window top: stored start values with k > 0 are <= 2^TWIN
#define SHT_SWIN 480      // window stride: true value = stored * 2^(-SWIN*k)
#define SHT_JCHK 8        // steps between window checks
#define SHT_TQ 16         // quantum of the kappa tables: one row per l_top multiple of TQ

struct ThetaPass {
    int n;                 // second index of d^l_{m,n} in this pass
    int sgn_out;           // harmonic order served at recursion step m is m_out = sgn_out * m  (P mode)
    int m_end;             // last recursion step (inclusive), <= 0
    int slab;              // which (n-)slab of the in/out arrays this pass belongs to
    const double* st_val;  // [Lp][ntp] windowed start values of d^l_{l,n}
    const uint8_t* st_k;   // [Lp][ntp] window counters
    const int* m_lo;       // [ntp] ring theta is served at step m iff m >= m_lo[theta] (nullptr: always)
    const double2* in;     // inverse: G[m-m_end][Lp][NC]   forward: W[m-m_end][ntp][NC]
    double2* out;          // inverse: F[row][ntp] (row = m_out mod NB)   forward: H[m_out+L-1][Lp]
};

struct ThetaArgs {
    int L, Lp;             // band-limit, padded (multiple of 128)
    int nth, ntp;          // regular rings, padded (multiple of 128)
    int NB;                // rows of the inverse output (FFT length in phi, 2L-1 on MW)
    const double* csc;     // [ntp] 1/sin(theta)
    const double* tau;     // [ntp] +tan(theta/2) (north) or -cot(theta/2) (south)
    const double* sig;     // [ntp] +1 north, -1 south
    const int8_t* kexp;    // [Lp/TQ][kstride] kappa exponents, column m - kmin
    int kstride, kmin;
    const double* rsq;     // [2*Lp+64] 1/sqrt(k)
    const ThetaPass* passes;
    int npass;
    int all_n_zero;        // every pass of this launch has n == 0 (lets the kernel use lambda' = -m cot(theta) S_m)
};

// launchers (theta_kernels.cu); mode 0 = PM (spin 0 complex: +m and -m from one pass), 1 = P (one order per step)
cudaError_t launch_theta_inverse(const ThetaArgs& a, int mode, cudaStream_t st);
cudaError_t launch_theta_forward(const ThetaArgs& a, int mode, cudaStream_t st);
cudaError_t launch_fp64_peak(int iters, double* sink, cudaStream_t st, int* blocks, int* threads, int* fma_per_thread);

void count_launch(int n = 1);
