// noalloc.cu -- s2_theta_inverse_noalloc: the theta step of the inverse transform (Eq. 33) for callers that cannot
// allocate (code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc).  No plan, no workspace, no
// cudaMalloc / cudaFree / cuFFT: a variant of the stored-table kernels of precompute.cu (the paper's precompute mode, Sec. 4.3,
// PAPER.md:411-419) whose d-function table lives in ONE file-scope device array of fixed size:
//   kernel 1 (na_fill_kernel)     d^l_{m,-s}(theta_t) of every degree, order and ring -> table E[m + L - 1][t][l]   (Eq. 25-29)
//   kernel 2 (na_inverse_kernel)  F_m(theta_t) = (-1)^s sum_l sqrt((2l+1)/4pi) E[m][t][l] flm[l][m]                 (Eq. 33)
// The table is SHT_NOALLOC_SCRATCH_BYTES (8 MiB) on every GPU that loads the library, held until the process exits; a request
// needs (2L-1) * ntheta * L doubles of it and is refused with a clear error beyond that (L = 64 on 2L rings fits; L = 80 on L rings).
// Every call shares the table: kernel 1 rewrites every entry the call's kernel 2 reads (zeros included), so nothing of the last
// call survives into this one; two calls that overlap on the GPU (different streams, no event between them) race on it.
//
// The recursion is the paper's, written out plainly (this path is for small L, not for speed): Eq. 27 start value as a product with
// a running power-of-two exponent, Eq. 25 down in m with the iterates rescaled by powers of two whenever they leave [2^-256, 2^256]
// (exact), and the two passes of DESIGN.md R5 -- second index n = -s serves the orders m >= m_s = round(n cos theta), second index
// -n serves the rest through d^l_{m,n} = (-1)^{m-n} d^l_{-m,-n} -- so that no iterate is used past the peak of its sequence.
// Rings within 1e-12 of a pole take the closed forms of Eq. 28 / 29.
#include "../../include/b200sht.h"
#include "internal.h"

#include <cuda_runtime.h>
#include <math.h>
#include <stdio.h>

#include <mutex>

namespace {

constexpr size_t NA_MAX_DOUBLES = SHT_NOALLOC_SCRATCH_BYTES / sizeof(double);
constexpr int NA_MAX_DEVICES = 64;

// The scratch.  In host code this name is a stand-in, not a device address: the host takes its address once per device with
// cudaGetSymbolAddress (na_scratch_ptr below) and passes that pointer to the kernels.
static __device__ __align__(256) double g_na_scratch[NA_MAX_DOUBLES];

struct NaArgs {
    int L, spin, ntheta;
    double* E;                                  // [2L-1][ntheta][L]
    const double2* flm;                         // [L][2L-1]
    double2* Fm;                                // [2L-1][ntheta]
    double theta[SHT_NOALLOC_MAX_RINGS];
};

// value = mant * 2^ex with |mant| in [1/2, 1)
__device__ __forceinline__ void na_norm(double& mant, int& ex) {
    int e; mant = frexp(mant, &e); ex += e;
}

// Eq. 27: d^l_{l,n}(beta) = sqrt((2l)! / ((l+n)! (l-n)!)) (-sin(beta/2))^{l-n} cos(beta/2)^{l+n}; the square root is the binomial
// coefficient C(2l, l+n) = prod_{j=1..l-n} (l+n+j)/j
__device__ void na_seed(int l, int n, double sh, double ch, double& mant, int& ex) {
    mant = 1.0; ex = 0;
    for (int j = 1; j <= l - n; ++j) { mant *= sqrt((double)(l + n + j) / (double)j) * (-sh); na_norm(mant, ex); }
    for (int j = 1; j <= l + n; ++j) { mant *= ch; na_norm(mant, ex); }
}

// Eq. 25 / 26 from m = l down to m_stop (>= -l) with second index n; the iterate of step m is stored at order flip * m:
//   flip = +1: E[m] = d^l_{m,n}                      (pass A)
//   flip = -1: E[-m] = (-1)^{m+n} d^l_{m,n}         (pass B: d^l_{-m,-n} = (-1)^{m-n} d^l_{m,n}, called with the negated index)
__device__ void na_recurse(int l, int n, int m_stop, int flip, double sh, double ch, double* E, size_t mstride, int L) {
    const double sinb = 2.0 * sh * ch, cosb = ch * ch - sh * sh;
    double cur, prev = 0.0; int ex;
    na_seed(l, n, sh, ch, cur, ex);
    for (int m = l; m >= m_stop; --m) {
        double v = scalbn(cur, ex);
        if (flip < 0 && ((m + n) & 1)) v = -v;
        E[(size_t)(flip * m + L - 1) * mstride] = v;
        if (m == m_stop) break;
        // d_{m-1} = a_{m-1} (lambda_m d_m - d_{m+1} / a_m),  2 / a_m = sqrt((l-m)(l+m+1))  (0 at m = l, where d_{l+1} = 0)
        const double lam = ((double)n - (double)m * cosb) / sinb;
        const double inv_am = 0.5 * sqrt((double)(l - m) * (double)(l + m + 1));
        const double am1 = 2.0 / sqrt((double)(l - m + 1) * (double)(l + m));
        const double nxt = am1 * (lam * cur - inv_am * prev);
        prev = cur; cur = nxt;
        const double a = fabs(cur);
        if (a != 0.0 && (a > 0x1p256 || a < 0x1p-256)) {
            const int e = ilogb(cur);
            cur = scalbn(cur, -e); prev = scalbn(prev, -e); ex += e;
        }
    }
}

// one thread per (degree l, ring t): every order m of the table column, zeros where |m| > l or l < |s|
__global__ void __launch_bounds__(256) na_fill_kernel(const NaArgs A) {
    const int l = blockIdx.x * 32 + threadIdx.x, t = blockIdx.y * 8 + threadIdx.y;
    if (l >= A.L || t >= A.ntheta) return;
    const int L = A.L, n = -A.spin, an = n < 0 ? -n : n;
    const size_t mstride = (size_t)A.ntheta * L;
    double* E = A.E + (size_t)t * L + l;                      // E[(m + L - 1) * mstride]
    for (int mi = 0; mi < 2 * L - 1; ++mi) {                  // clear what the passes below do not write
        const int m = mi - (L - 1), am = m < 0 ? -m : m;
        if (am > l || l < an) E[(size_t)mi * mstride] = 0.0;
    }
    if (l < an) return;
    const double beta = A.theta[t];
    const double pi = 3.14159265358979323846;
    if (beta <= 1e-12 || pi - beta <= 1e-12) {                // Eq. 28: d(0) = delta_{mn};  Eq. 29: d(pi) = (-1)^{l+m} delta_{m,-n}
        const bool north = beta <= 1e-12;
        for (int m = -l; m <= l; ++m) {
            double v = 0.0;
            if (north && m == n) v = 1.0;
            if (!north && m == -n) v = ((l + m) & 1) ? -1.0 : 1.0;
            E[(size_t)(m + L - 1) * mstride] = v;
        }
        return;
    }
    const double sh = sin(0.5 * beta), ch = cos(0.5 * beta);
    const int ms = (int)rint((double)n * (ch * ch - sh * sh));      // |ms| <= |n| <= l
    na_recurse(l, n, ms, +1, sh, ch, E, mstride, L);                // orders m in [ms, l]
    if (1 - ms <= l) na_recurse(l, -n, 1 - ms, -1, sh, ch, E, mstride, L);   // orders m' in [1 - ms, l] of index -n = orders -m' of index n
}

// one warp per (order m, ring t), lanes over the degrees; writes F_m(theta_t) (no atomics: the output needs no clearing)
constexpr int NA_WARPS = 8;
__global__ void __launch_bounds__(NA_WARPS * 32) na_inverse_kernel(const NaArgs A) {
    const int L = A.L, mi = blockIdx.y, m = mi - (L - 1);
    const int lane = threadIdx.x & 31, t = blockIdx.x * NA_WARPS + (threadIdx.x >> 5);
    if (t >= A.ntheta) return;
    const int an = A.spin < 0 ? -A.spin : A.spin, am = m < 0 ? -m : m, l_lo = am > an ? am : an;
    const double* E = A.E + ((size_t)mi * A.ntheta + t) * L;
    double re = 0.0, im = 0.0;
    for (int l = l_lo + lane; l < L; l += 32) {
        const double p = E[l] * sqrt((double)(2 * l + 1) / (4.0 * 3.14159265358979323846));
        const double2 c = A.flm[(size_t)l * (2 * L - 1) + mi];
        re = fma(p, c.x, re); im = fma(p, c.y, im);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) { re += __shfl_xor_sync(0xffffffffu, re, o); im += __shfl_xor_sync(0xffffffffu, im, o); }
    if (lane == 0) {
        const double sg = (A.spin & 1) ? -1.0 : 1.0;
        A.Fm[(size_t)mi * A.ntheta + t] = make_double2(sg * re, sg * im);
    }
}

// device address of the scratch on the current device, looked up once per device
cudaError_t na_scratch_ptr(double** out) {
    static std::mutex mu;
    static double* ptr[NA_MAX_DEVICES] = {};
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= NA_MAX_DEVICES) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(mu);
    if (!ptr[dev]) {
        double* p = nullptr;
        e = cudaGetSymbolAddress((void**)&p, g_na_scratch);
        if (e != cudaSuccess) return e;
        ptr[dev] = p;
    }
    *out = ptr[dev];
    return cudaSuccess;
}

sht_status na_fail(sht_status s, char* err, size_t err_len, const char* msg) {
    if (err && err_len) snprintf(err, err_len, "%s", msg);
    return s;
}

}  // namespace

extern "C" sht_status s2_theta_inverse_noalloc(int L, int spin, int ntheta, const double* theta, const void* flm, void* Fm,
                                               sht_stream stream, char* err, size_t err_len) {
    char msg[256];
    if (err && err_len) err[0] = 0;
    if (L < 1 || spin <= -L || spin >= L) return na_fail(SHT_EINVAL, err, err_len, "s2_theta_inverse_noalloc: need L >= 1 and |spin| < L");
    if (!theta || !flm || !Fm) return na_fail(SHT_EINVAL, err, err_len, "s2_theta_inverse_noalloc: null pointer");
    if (ntheta < 1 || ntheta > SHT_NOALLOC_MAX_RINGS) {
        snprintf(msg, sizeof msg, "s2_theta_inverse_noalloc: ntheta = %d outside 1..%d (SHT_NOALLOC_MAX_RINGS)", ntheta, SHT_NOALLOC_MAX_RINGS);
        return na_fail(SHT_EUNSUPPORTED, err, err_len, msg);
    }
    const size_t need = (size_t)(2 * L - 1) * (size_t)ntheta * (size_t)L;
    if (need > NA_MAX_DOUBLES) {
        snprintf(msg, sizeof msg, "s2_theta_inverse_noalloc: (2L-1) * ntheta * L = %zu table entries exceed the fixed scratch of %zu "
                 "(SHT_NOALLOC_SCRATCH_BYTES = %d); use a plan (s2_theta_inverse_plan) for this size", need, (size_t)NA_MAX_DOUBLES,
                 (int)SHT_NOALLOC_SCRATCH_BYTES);
        return na_fail(SHT_EUNSUPPORTED, err, err_len, msg);
    }
    NaArgs a;
    a.L = L; a.spin = spin; a.ntheta = ntheta;
    for (int t = 0; t < ntheta; ++t) {
        if (!(theta[t] >= 0.0 && theta[t] <= 3.14159265358979323846 + 1e-12))
            return na_fail(SHT_EINVAL, err, err_len, "s2_theta_inverse_noalloc: ring colatitudes must lie in [0, pi]");
        a.theta[t] = theta[t];
    }
    cudaError_t e = na_scratch_ptr(&a.E);
    if (e != cudaSuccess) {
        snprintf(msg, sizeof msg, "s2_theta_inverse_noalloc: cudaGetSymbolAddress(scratch): %s", cudaGetErrorString(e));
        return na_fail(SHT_ECUDA, err, err_len, msg);
    }
    a.flm = static_cast<const double2*>(flm);
    a.Fm = static_cast<double2*>(Fm);
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    na_fill_kernel<<<dim3((L + 31) / 32, (ntheta + 7) / 8), dim3(32, 8), 0, st>>>(a);
    na_inverse_kernel<<<dim3((ntheta + NA_WARPS - 1) / NA_WARPS, 2 * L - 1), NA_WARPS * 32, 0, st>>>(a);
    count_launch(2);
    e = cudaGetLastError();
    if (e != cudaSuccess) {
        snprintf(msg, sizeof msg, "s2_theta_inverse_noalloc: kernel launch: %s", cudaGetErrorString(e));
        return na_fail(SHT_ECUDA, err, err_len, msg);
    }
    return SHT_OK;
}
