// precompute.cu -- the paper's "full precomputation" mode (Sec. 4.3): the Wigner d-functions d^l_{m,-s}(theta) of
// every degree, order and ring are computed once, stored (O(L^3) memory), and the theta step of Eq. 30 / 33 becomes a plain
// weighted sum -- the einsum 'tlm,tm->lm' of PAPER.md:419.  On a B200 this pays at moderate band-limits (L <= 512), where the
// on-the-fly kernels are bound by the latency of their L sequential recursion steps while the stored table streams from HBM / L2;
// at larger L the O(L^3) table is slower to read than the d-functions are to recompute, which is why on-the-fly is the default.
//
// What is stored is exactly what the on-the-fly kernels hold in registers at recursion step m: the "e-form" iterate
// e^l_m(theta) = d^l_{m,n}(theta) / c_m(l) (internal.h), produced by the same recursion (Eq. 25-27) with the same tables, so that
// the operand tables of the on-the-fly path (G with c_m(l) folded in, W, ctab) serve both modes:
//   E[pass][m - m_end][ring][l]   (l fastest; 0 where l < max(|m|, |n|), where the ring is not served by the pass (peak split,
//                                  DESIGN.md R5) or where the true value is below 2^-340)
//   inverse  F[row(m_out)][ring] += sum_l     E[m][ring][l] * G[m][l]            (warp per ring, lanes over l)
//   forward  H[m_out+L-1][l]     += c_m(l) * sum_ring E[m][ring][l] * W[m][ring]   (thread per l, loop over rings)
// Both transform kernels are HBM-bound: they read E once (triangular part only).
#include "device_utils.cuh"
#include "internal.h"

#include <cuda_runtime.h>
#include <stdint.h>

namespace {

using namespace shtdev;

// ---- table fill: one thread per (l, ring), sequential in m (plan time) -----------------------------------------------------
__global__ void __launch_bounds__(256) pre_fill_kernel(const ThetaArgs A) {
    const ThetaPass P = A.passes[blockIdx.z];
    const int l = blockIdx.x * 32 + threadIdx.x, th = blockIdx.y * 8 + threadIdx.y;
    const int an = P.n < 0 ? -P.n : P.n;
    if (l >= A.L || l < an || th >= A.nth) return;
    const int m_end = P.m_end;
    const int mlo = P.m_lo ? max(P.m_lo[th], m_end) : m_end;
    double cur = P.st_val[(size_t)l * A.ntp + th], prev = 0.0;
    int k = P.st_k[(size_t)l * A.ntp + th];
    const double2* sg = A.sg + (size_t)(l / SHT_TQ) * A.sgstride - A.mmin;
    double* E = const_cast<double*>(P.pre);
    const double shift = pow2i(-SHT_SWIN);
    double x = 0.0;                                    // (l - m)(l + m + 1), 0 at m = l
    for (int m = l; m >= mlo; --m) {
        E[((size_t)(m - m_end) * A.ntp + th) * A.Lp + l] = k == 0 ? cur : 0.0;
        if (m == mlo) break;
        const double2 c = sg[m];
        const double lam = P.lam[(size_t)(m - m_end + 1) * A.ntp + th] * c.x;
        const double nxt = fma(lam, cur, -((x * c.y) * prev));
        prev = cur; cur = nxt;
        x += 2.0 * (double)m;                          // x_{m-1} = x_m + 2m
        if (k > 0 && hi_abs(cur) > SHT_HI_TWIN) { cur *= shift; prev *= shift; --k; }
    }
}

// ---- inverse, Eq. 33 with stored d-functions ----------------------------------------------------------------------------------
constexpr int PI_WARPS = 8;                            // rings per block (one warp each)
template <int NC>
__global__ void __launch_bounds__(PI_WARPS * 32) pre_inverse_kernel(const ThetaArgs A) {
    constexpr int ROWD = 2 * NC + 2;
    const ThetaPass P = A.passes[blockIdx.z];
    const int m = A.L - 1 - (int)blockIdx.y, m_end = P.m_end;
    if (m < m_end) return;
    const int an = P.n < 0 ? -P.n : P.n, am = m < 0 ? -m : m, l_lo = am > an ? am : an;
    const int lane = threadIdx.x & 31, th = blockIdx.x * PI_WARPS + (threadIdx.x >> 5);
    if (l_lo >= A.L || th >= A.nth || th < A.th_lo || th >= A.th_hi) return;
    if (P.m_lo && m < P.m_lo[th]) return;
    const double* E = P.pre + ((size_t)(m - m_end) * A.ntp + th) * A.Lp;
    const double* G = P.in + (size_t)(m - m_end + 1) * A.Lp * ROWD;
    double acc[2 * NC];
#pragma unroll
    for (int c = 0; c < 2 * NC; ++c) acc[c] = 0.0;
    for (int l = (l_lo & ~31) + lane; l < A.L; l += 32) {
        const double e = E[l];
        const double* r = G + (size_t)l * ROWD;
#pragma unroll
        for (int c = 0; c < 2 * NC; ++c) acc[c] = fma(e, r[c], acc[c]);
    }
#pragma unroll
    for (int c = 0; c < 2 * NC; ++c)
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) acc[c] += __shfl_xor_sync(0xffffffffu, acc[c], o);
    if (lane == 0) {
        double* out = reinterpret_cast<double*>(P.out) + (size_t)th * 2;
#pragma unroll
        for (int c = 0; c < NC; ++c) {
            if (c == 1 && m == 0) continue;
            const int m_out = (NC == 2) ? (c ? -m : m) : P.sgn_out * m;
            const int row = m_out < 0 ? m_out + A.NB : m_out;
            double* o = out + (size_t)row * A.ldout * 2;
            red_add_f64(o, acc[2 * c]); red_add_f64(o + 1, acc[2 * c + 1]);
        }
    }
}

// ---- forward, Eq. 30 with stored d-functions ----------------------------------------------------------------------------------
constexpr int PF_T = 128;                              // degrees per block = rings per shared-memory chunk
constexpr int PF_SPLIT = 4;                            // blocks sharing the rings of one (degree tile, m): more parallelism at moderate L
template <int NC>
__global__ void __launch_bounds__(PF_T) pre_forward_kernel(const ThetaArgs A) {
    __shared__ double2 sw[PF_T][NC];
    const ThetaPass P = A.passes[blockIdx.z];
    const int m = A.L - 1 - (int)blockIdx.y, m_end = P.m_end;
    if (m < m_end) return;
    const int an = P.n < 0 ? -P.n : P.n, am = m < 0 ? -m : m, l_lo = am > an ? am : an;
    const int l0 = (blockIdx.x / PF_SPLIT) * PF_T, l = l0 + threadIdx.x, part = blockIdx.x % PF_SPLIT;
    if (l0 + PF_T <= l_lo || l0 >= A.L) return;
    const double* E = P.pre + (size_t)(m - m_end) * A.ntp * A.Lp;
    const double2* W = reinterpret_cast<const double2*>(P.in) + (size_t)(m - m_end + 1) * A.ntp * NC;
    double acc[4][2 * NC];
#pragma unroll
    for (int u = 0; u < 4; ++u)
#pragma unroll
        for (int c = 0; c < 2 * NC; ++c) acc[u][c] = 0.0;
    // this block's share of the (shard's) rings, in chunks of PF_T
    const int r_lo = A.th_lo, r_hi = min(A.th_hi, A.nth);
    const int per = ((r_hi - r_lo + PF_SPLIT - 1) / PF_SPLIT + 3) & ~3;
    const int t_lo = r_lo + part * per, t_hi = min(r_hi, t_lo + per);
    for (int t0 = t_lo; t0 < t_hi; t0 += PF_T) {
        __syncthreads();
        const int tt = t0 + threadIdx.x;
#pragma unroll
        for (int c = 0; c < NC; ++c) sw[threadIdx.x][c] = tt < t_hi ? W[(size_t)tt * NC + c] : make_double2(0.0, 0.0);
        __syncthreads();
        const int nt = min(PF_T, t_hi - t0);
        const double* e = E + (size_t)t0 * A.Lp + l;
        for (int t = 0; t < nt; t += 4) {              // (rows beyond nt inside the chunk carry zero weights; E is allocated to ntp rows)
            double ev[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) ev[u] = t0 + t + u < A.ntp ? e[(size_t)(t + u) * A.Lp] : 0.0;
#pragma unroll
            for (int u = 0; u < 4; ++u)
#pragma unroll
                for (int c = 0; c < NC; ++c) {
                    acc[u][2 * c] = fma(ev[u], sw[t + u][c].x, acc[u][2 * c]); acc[u][2 * c + 1] = fma(ev[u], sw[t + u][c].y, acc[u][2 * c + 1]);
                }
        }
    }
    if (l < an || l >= A.L || l < m || l < -m) return;
    const double cm = A.ctab[(size_t)(m - A.mmin) * A.Lp + l];
#pragma unroll
    for (int c = 0; c < NC; ++c) {
        const bool neg = NC == 2 && c == 1;
        const int m_out = (NC == 2) ? (neg ? -m : m) : P.sgn_out * m;
        const double f = (P.fold && neg && ((l - P.n) & 1)) ? -cm : cm;          // (-1)^{l-n} on the mirrored-ring column of a fold pass
        double* o = reinterpret_cast<double*>(P.out) + ((size_t)(m_out + A.L - 1) * A.Lp + l) * 2;
        red_add_f64(o, ((acc[0][2 * c] + acc[1][2 * c]) + (acc[2][2 * c] + acc[3][2 * c])) * f);
        red_add_f64(o + 1, ((acc[0][2 * c + 1] + acc[1][2 * c + 1]) + (acc[2][2 * c + 1] + acc[3][2 * c + 1])) * f);
    }
}

}  // namespace

cudaError_t launch_pre_fill(const ThetaArgs& a, cudaStream_t st) {
    if (a.npass == 0 || a.nth == 0) return cudaSuccess;
    dim3 grid((a.L + 31) / 32, (a.nth + 7) / 8, a.npass), block(32, 8);
    pre_fill_kernel<<<grid, block, 0, st>>>(a);
    count_launch();
    return cudaGetLastError();
}
cudaError_t launch_pre_inverse(const ThetaArgs& a, int mode, int nrows, cudaStream_t st) {
    if (a.npass == 0 || a.nth == 0) return cudaSuccess;
    dim3 grid((a.nth + PI_WARPS - 1) / PI_WARPS, nrows, a.npass);
    if (mode == 0) pre_inverse_kernel<2><<<grid, PI_WARPS * 32, 0, st>>>(a);
    else pre_inverse_kernel<1><<<grid, PI_WARPS * 32, 0, st>>>(a);
    count_launch();
    return cudaGetLastError();
}
cudaError_t launch_pre_forward(const ThetaArgs& a, int mode, int nrows, cudaStream_t st) {
    if (a.npass == 0 || a.nth == 0) return cudaSuccess;
    dim3 grid((a.Lp / PF_T) * PF_SPLIT, nrows, a.npass);
    if (mode == 0) pre_forward_kernel<2><<<grid, PF_T, 0, st>>>(a);
    else pre_forward_kernel<1><<<grid, PF_T, 0, st>>>(a);
    count_launch();
    return cudaGetLastError();
}
