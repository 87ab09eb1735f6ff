// healpix.cu -- HEALPix ring Fourier staging (Sec. 4.2.4): per-ring DFTs of variable length with the
// ring's phi offset applied as a phase and F_m periodically extended (forward) / folded (inverse) in m (R13):
//   forward  F_m(theta_r) = e^{-i m phi0(r)} X_r[m mod nphi(r)],   X_r = DFT_nphi(f_r)
//   inverse  Y_r[k] = sum_{m = k mod nphi} F_m(theta_r) e^{+i m phi0(r)},   f_r = nphi-point synthesis of Y_r.
// The 2 nside+1 belt rings (nphi = 4 nside, contiguous in the ring-ordered map) go through one batched cuFFT call.
// The 2 (nside-1) polar-cap rings have nside-1 distinct lengths 4r; they are all transformed at ONE power-of-two
// length M >= 2*4(nside-1)-1 by Bluestein's chirp-z identity  jk = (j^2 + k^2 - (k-j)^2)/2:
//   X_k = conj(b_k) * sum_j (x_j conj(b_j)) b_{k-j},   b_j = e^{i pi j^2 / n},
// i.e. one batched M-point cuFFT, a pointwise product with the precomputed FFT of the chirp, one batched inverse.
// HBM-bound staging, timed apart from the hot path.
#include "staging.h"

#include <math.h>

namespace {

struct HpRing { int n; int shifted; long long off; int cap; };   // cap: index into the Bluestein batch, or -1 (belt)

// ring i = 0..4 nside-2 (north to south), public HEALPix ring scheme (R11)
__host__ __device__ inline HpRing hp_ring(int nside, int i) {
    HpRing g;
    const int r = i + 1, rr = r <= 2 * nside ? r : 4 * nside - r;
    const long long npix = 12LL * nside * nside;
    if (rr < nside) {
        g.n = 4 * rr; g.shifted = 1;
        g.off = r <= 2 * nside ? 2LL * rr * (rr - 1) : npix - 2LL * rr * (rr + 1);
        g.cap = r <= 2 * nside ? rr - 1 : (nside - 1) + (rr - 1);
    } else {
        g.n = 4 * nside; g.shifted = ((rr - nside) & 1) == 0;
        g.off = 2LL * nside * (nside - 1) + (long long)(r - nside) * 4 * nside;
        g.cap = -1;
    }
    return g;
}
// b_j = e^{i pi j^2/n} with j^2 reduced mod 2n in integers
__device__ __forceinline__ double2 chirp(long long j, int n) {
    long long q = (j * j) % (2LL * n);
    double s, c;
    sincospi((double)q / (double)n, &s, &c);
    return make_double2(c, s);
}
__device__ __forceinline__ double2 cmul(double2 a, double2 b) { return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }
__device__ __forceinline__ double2 cmulc(double2 a, double2 b) { return make_double2(a.x * b.x + a.y * b.y, a.y * b.x - a.x * b.y); }   // a * conj(b)

// chirp filter of cap length n = 4(c+1), c < nside-1: row c of BF, wrapped to length M, scaled 1/M (FFT applied afterwards)
__global__ void k_hp_chirp(int nside, int M, double2* __restrict__ BF) {
    const int c = blockIdx.y, j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= M) return;
    const int n = 4 * (c + 1);
    double2 v = make_double2(0.0, 0.0);
    int d = j < n ? j : (j > M - n ? M - j : -1);
    if (d >= 0) { v = chirp(d, n); v.x /= (double)M; v.y /= (double)M; }
    BF[(size_t)c * M + j] = v;
}
// forward pack: cap ring samples times conj(b_j), zero padded.  real_in: the map is an array of doubles.
__global__ void k_hp_pack_fwd(int nside, int M, int real_in, const void* __restrict__ map, double2* __restrict__ C) {
    const int c = blockIdx.y, j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= M) return;
    const int north = c < nside - 1, rr = north ? c + 1 : c - (nside - 1) + 1;
    const HpRing g = hp_ring(nside, north ? rr - 1 : 4 * nside - rr - 1);
    double2 v = make_double2(0.0, 0.0);
    if (j < g.n) {
        double2 x = real_in ? make_double2(((const double*)map)[g.off + j], 0.0) : ((const double2*)map)[g.off + j];
        v = cmulc(x, chirp(j, g.n));
    }
    C[(size_t)c * M + j] = v;
}
// pointwise product with the chirp spectrum (row shared by the north and the south ring of the same length)
__global__ void k_hp_mul(int nside, int M, const double2* __restrict__ BF, double2* __restrict__ C) {
    const int c = blockIdx.y, j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= M) return;
    const int cb = c < nside - 1 ? c : c - (nside - 1);
    C[(size_t)c * M + j] = cmul(C[(size_t)c * M + j], BF[(size_t)cb * M + j]);
}
// forward unpack: U[bin(m)][ring] = wphase * X_ring[m mod n],  m = mlo..L-1 (bin = m mod NB), through a 32x32 transpose
__global__ void k_hp_unpack_fwd(int nside, int L, int NB, int mlo, int nth, int ldu, int M, const double2* __restrict__ C,
                                const double2* __restrict__ E, double2* __restrict__ U) {
    __shared__ double2 tile[32][33];
    const int i0 = blockIdx.x * 32, m0 = mlo + blockIdx.y * 32;
    for (int q = threadIdx.y; q < 32; q += blockDim.y) {          // rows: rings; columns: m (contiguous bins of one ring)
        const int i = i0 + q, m = m0 + threadIdx.x;
        double2 v = make_double2(0.0, 0.0);
        if (i < nth && m < L) {
            const HpRing g = hp_ring(nside, i);
            int k = m % g.n; if (k < 0) k += g.n;
            double2 x;
            if (g.cap >= 0) x = cmulc(C[(size_t)g.cap * M + k], chirp(k, g.n));
            else x = E[(size_t)(i - (nside - 1)) * g.n + k];
            if (g.shifted) {                                       // e^{-i m pi/n}
                long long r = ((long long)m) % (2LL * g.n); if (r < 0) r += 2LL * g.n;
                double s, c; sincospi((double)r / (double)g.n, &s, &c);
                x = cmulc(x, make_double2(c, s));
            }
            v = x;
        }
        tile[q][threadIdx.x] = v;
    }
    __syncthreads();
    for (int q = threadIdx.y; q < 32; q += blockDim.y) {
        const int m = m0 + q, i = i0 + threadIdx.x;
        if (m < L && i < nth) U[(size_t)(m < 0 ? m + NB : m) * ldu + i] = tile[threadIdx.x][q];
    }
}
// inverse fold: Y_ring[k] = sum_{m = k mod n, |m| < L} F[bin(m)][ring] e^{+i m phi0}.  Cap rings go into the Bluestein batch as
// conj(Y_k) conj(b_k) (synthesis = conj(DFT(conj Y))), belt rings into E.  F is bin-major (rows m, rings contiguous) and the targets are
// ring-major, so a 32 x 32 tile is read along the rings and, transposed through shared memory, added along k: C and E are zeroed
// first and every term is added with RED.ADD.F64 (the map is linear; several m fold onto one k wherever n < 2L-1).
__global__ void k_hp_fold_inv(int nside, int L, int NB, int nth, int ldf, int M, const double2* __restrict__ F,
                              double2* __restrict__ C, double2* __restrict__ E) {
    __shared__ double2 tile[32][33];
    const int i0 = blockIdx.x * 32, mi0 = blockIdx.y * 32;        // mi = m + L - 1
    for (int q = threadIdx.y; q < 32; q += blockDim.y) {
        const int mi = mi0 + q, i = i0 + threadIdx.x, m = mi - (L - 1);
        double2 v = make_double2(0.0, 0.0);
        if (mi < 2 * L - 1 && i < nth) v = F[(size_t)(m < 0 ? m + NB : m) * ldf + i];
        tile[q][threadIdx.x] = v;
    }
    __syncthreads();
    for (int q = threadIdx.y; q < 32; q += blockDim.y) {
        const int i = i0 + q, mi = mi0 + threadIdx.x, m = mi - (L - 1);
        if (i >= nth || mi >= 2 * L - 1) continue;
        const HpRing g = hp_ring(nside, i);
        double2 x = tile[threadIdx.x][q];
        int k = m % g.n; if (k < 0) k += g.n;
        if (g.shifted) {
            long long r = ((long long)m) % (2LL * g.n); if (r < 0) r += 2LL * g.n;
            double s, c; sincospi((double)r / (double)g.n, &s, &c);
            x = cmul(x, make_double2(c, s));
        }
        double* dst;
        if (g.cap >= 0) { x = cmulc(make_double2(x.x, -x.y), chirp(k, g.n)); dst = reinterpret_cast<double*>(C + (size_t)g.cap * M + k); }
        else dst = reinterpret_cast<double*>(E + (size_t)(i - (nside - 1)) * g.n + k);
        asm volatile("red.global.add.f64 [%0], %1;" ::"l"(dst), "d"(x.x) : "memory");
        asm volatile("red.global.add.f64 [%0], %1;" ::"l"(dst + 1), "d"(x.y) : "memory");
    }
}
// inverse unpack of the cap rings: f_j = conj( conj(b_j) * conv_j ) = b_j * conj(conv_j)
__global__ void k_hp_unpack_inv(int nside, int M, int real_out, const double2* __restrict__ C, void* __restrict__ map) {
    const int c = blockIdx.y, j = blockIdx.x * blockDim.x + threadIdx.x;
    const int north = c < nside - 1, rr = north ? c + 1 : c - (nside - 1) + 1;
    const HpRing g = hp_ring(nside, north ? rr - 1 : 4 * nside - rr - 1);
    if (j >= g.n) return;
    double2 y = C[(size_t)c * M + j];
    double2 v = cmul(chirp(j, g.n), make_double2(y.x, -y.y));
    if (real_out) ((double*)map)[g.off + j] = v.x;
    else ((double2*)map)[g.off + j] = v;
}
// belt rings, real maps: real part of the synthesised rows
__global__ void k_hp_belt_real(size_t n, const double2* __restrict__ E, double* __restrict__ out) {
    size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) out[i] = E[i].x;
}

inline unsigned cdiv(size_t a, size_t b) { return (unsigned)((a + b - 1) / b); }

}  // namespace

#define LAUNCHED() do { count_launch(); cudaError_t e_ = cudaGetLastError(); if (e_ != cudaSuccess) return e_; } while (0)

void hp_ring_host(int nside, int i, int* nphi, int* shifted, long long* off) {
    HpRing g = hp_ring(nside, i);
    *nphi = g.n; *shifted = g.shifted; *off = g.off;
}
cudaError_t st_hp_chirp(int nside, int M, double2* BF, cudaStream_t st) {
    if (nside < 2) return cudaSuccess;
    k_hp_chirp<<<dim3(cdiv(M, 256), nside - 1), 256, 0, st>>>(nside, M, BF);
    LAUNCHED(); return cudaSuccess;
}
cudaError_t st_hp_pack_fwd(int nside, int M, int real_in, const void* map, double2* C, cudaStream_t st) {
    if (nside < 2) return cudaSuccess;
    k_hp_pack_fwd<<<dim3(cdiv(M, 256), 2 * (nside - 1)), 256, 0, st>>>(nside, M, real_in, map, C);
    count_bytes(16.0 * (double)M * 2 * (nside - 1) + 16.0 * 4.0 * (double)nside * (nside - 1)); LAUNCHED(); return cudaSuccess;
}
cudaError_t st_hp_mul(int nside, int M, const double2* BF, double2* C, cudaStream_t st) {
    if (nside < 2) return cudaSuccess;
    k_hp_mul<<<dim3(cdiv(M, 256), 2 * (nside - 1)), 256, 0, st>>>(nside, M, BF, C);
    count_bytes(48.0 * (double)M * 2 * (nside - 1)); LAUNCHED(); return cudaSuccess;
}
cudaError_t st_hp_unpack_fwd(int nside, int L, int NB, int mlo, int ldu, int M, const double2* C, const double2* E, double2* U,
                             cudaStream_t st) {
    const int nth = 4 * nside - 1;
    k_hp_unpack_fwd<<<dim3(cdiv(nth, 32), cdiv(L - mlo, 32)), dim3(32, 8), 0, st>>>(nside, L, NB, mlo, nth, ldu, M, C, E, U);
    count_bytes(16.0 * (double)nth * (L - mlo) + 16.0 * 12.0 * (double)nside * nside); LAUNCHED(); return cudaSuccess;
}
cudaError_t st_hp_fold_inv(int nside, int L, int NB, int ldf, int M, const double2* F, double2* C, double2* E, cudaStream_t st) {
    const int nth = 4 * nside - 1;
    const size_t cb = sizeof(double2) * (size_t)M * 2 * (nside > 1 ? nside - 1 : 0), eb = sizeof(double2) * 4 * (size_t)nside * (2 * nside + 1);
    cudaError_t e = cb ? cudaMemsetAsync(C, 0, cb, st) : cudaSuccess;
    if (e == cudaSuccess) e = cudaMemsetAsync(E, 0, eb, st);
    if (e != cudaSuccess) return e;
    k_hp_fold_inv<<<dim3(cdiv(nth, 32), cdiv(2 * L - 1, 32)), dim3(32, 8), 0, st>>>(nside, L, NB, nth, ldf, M, F, C, E);
    count_bytes(32.0 * (double)nth * (2 * L - 1) + (double)cb + (double)eb); LAUNCHED(); return cudaSuccess;
}
cudaError_t st_hp_unpack_inv(int nside, int M, int real_out, const double2* C, void* map, cudaStream_t st) {
    if (nside < 2) return cudaSuccess;
    k_hp_unpack_inv<<<dim3(cdiv(4 * (nside - 1), 128), 2 * (nside - 1)), 128, 0, st>>>(nside, M, real_out, C, map);
    count_bytes(16.0 * (double)M * 2 * (nside - 1) + 16.0 * 4.0 * (double)nside * (nside - 1)); LAUNCHED(); return cudaSuccess;
}
cudaError_t st_hp_belt_real(size_t n, const double2* E, double* out, cudaStream_t st) {
    k_hp_belt_real<<<cdiv(n, 256), 256, 0, st>>>(n, E, out);
    count_bytes(24.0 * (double)n); LAUNCHED(); return cudaSuccess;
}
