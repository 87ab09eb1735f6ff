// theta_f32.cu -- the fp32 variant of the hot path (BASELINE config 5: "fp64 and fp32"): Wigner-d recursion in m (Eq. 25-27,
// PAPER.md:225-234) fused with the contractions of Eq. 30 / Eq. 33, with iterates, coefficients and partial sums in fp32.
//
// The fp64 kernels run the recursion in the "e-form" (internal.h), whose factor c_m(l) spans up to 2^250 inside a 64-degree
// quantum -- outside the fp32 exponent range.  Here the recursion is the paper's own form on the true d-values,
//     d_{m-1} = (lambda_m A_m(l)) d_m - B_m(l) d_{m+1},   A_m = a_{m-1} = 2/sqrt((l-m+1)(l+m)),   B_m = a_{m-1}/a_m,
// (3 FP32 instructions per step) with fp32 tables A, B (plan time) and the renormalisation of Sec. 3.4 as
// power-of-two windows sized for fp32: true value = stored * 2^(-48 k); a stored value with k > 0 stays below 2^-43 (it grows by
// less than 2^21 per step and is checked every step against 2^-64), which is below fp32 resolution of the sums, so no masking.
// Arithmetic is PACKED: a thread's items come in pairs of neighbouring rings held as float2, and every multiply-add is one
// fma.rn.f32x2 / mul.f32x2 (SASS FFMA2 / FMUL2, sm_100+; __ffma2_rn, __fmul2_rn) -- 7 packed instructions per pair of items and step
// (4 projection + 3 recursion).  A packed instruction occupies the FP32 pipe for two cycles but one issue slot, which leaves every
// other issue slot to the loads, stores and bookkeeping that the one-instruction-per-cycle FP32 pipe otherwise has to share with them.
// Scope: second index n = 0 (spin-0 plans), MW sampling, one map.  Everything around the two kernels (FFTs, staging, the pole
// ring) is the fp64 code; the kernels read fp32 operand tables and add their block sums into the fp64 F / H arrays.
#include "internal.h"

#include <cuda_pipeline.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace {

constexpr int FW = 48;                 // window stride (bits)
constexpr int FTOP = -64;              // a stored value with k > 0 is rescaled once it exceeds 2^FTOP
constexpr int TLF = 64, NTF = 128;     // block tile: degrees x rings
constexpr int NWF = 8;                 // warps per block

__device__ __forceinline__ float pow2f(int e) { return __int_as_float((127 + e) << 23); }
__device__ __forceinline__ void red_add_f64(double* gptr, double v) {
    asm volatile("red.global.add.f64 [%0], %1;" ::"l"(gptr), "d"(v) : "memory");
}

// window counters of 32 items, 16 bits each
struct KPackF {
    uint32_t w[16];
    __device__ __forceinline__ void fill(uint32_t v) {
#pragma unroll
        for (int i = 0; i < 16; ++i) w[i] = v;
    }
    __device__ __forceinline__ void set(int idx, uint32_t k) {
        const int sh = (idx & 1) * 16;
        w[idx >> 1] = (w[idx >> 1] & ~(0xffffu << sh)) | (k << sh);
    }
    __device__ __forceinline__ uint32_t get(int idx) const { return (w[idx >> 1] >> ((idx & 1) * 16)) & 0xffffu; }
    __device__ __forceinline__ void dec(int idx) { w[idx >> 1] -= 1u << ((idx & 1) * 16); }
    __device__ __forceinline__ bool any_nonzero() const {
        uint32_t o = 0;
#pragma unroll
        for (int i = 0; i < 16; ++i) o |= w[i];
        return o != 0;
    }
};
// items are stored as float2 pairs: item q = component q & 1 of pair q >> 1
// `contrib` (probe instantiations only) is raised when an item reaches its last window: from then on it contributes to the sums
template <int NP, bool TRACK>
__device__ __forceinline__ void window_check_f(float2 (&cur)[NP], float2 (&prev)[NP], KPackF& kp, bool& contrib) {
    const float s = pow2f(-FW), top = pow2f(FTOP);
#pragma unroll
    for (int q = 0; q < NP; ++q) {
        if (fabsf(cur[q].x) > top && kp.get(2 * q) != 0u) { cur[q].x *= s; prev[q].x *= s; kp.dec(2 * q); if (TRACK && kp.get(2 * q) == 0u) contrib = true; }
        if (fabsf(cur[q].y) > top && kp.get(2 * q + 1) != 0u) { cur[q].y *= s; prev[q].y *= s; kp.dec(2 * q + 1); if (TRACK && kp.get(2 * q + 1) == 0u) contrib = true; }
    }
}
// probe: does any item of this thread matter yet?  One in its last window (k = 0) whose magnitude is still below 2^-40 adds less than fp32
// resolution of an O(1) sum by a factor 2^16: as silent as one with k > 0.  (Items that have not started hold 0.)
template <int NP>
__device__ __forceinline__ bool f32_matters(const float2 (&cur)[NP], const KPackF& kp) {
    const float thr = pow2f(-40);
    bool big = false;
#pragma unroll
    for (int q = 0; q < NP; ++q)
        big = big || (kp.get(2 * q) == 0u && fabsf(cur[q].x) > thr) || (kp.get(2 * q + 1) == 0u && fabsf(cur[q].y) > thr);
    return big;
}
// ---- silent-head skip (internal.h ThetaArgs::skip_*): the state of a block at pair p0, thread-minor
template <int NP>
__device__ __forceinline__ void f32_state_store(const F32Args& A, int tid, const float2 (&cur)[NP], const float2 (&prev)[NP], const KPackF& kp) {
    float* d = reinterpret_cast<float*>(reinterpret_cast<char*>(A.skip_state) + (size_t)blockIdx.x * SHT_SKIP_STATE_BYTES_F32);
    uint32_t* u = reinterpret_cast<uint32_t*>(d + 64 * 256);
#pragma unroll
    for (int q = 0; q < NP; ++q) {
        d[(2 * q) * 256 + tid] = cur[q].x; d[(2 * q + 1) * 256 + tid] = cur[q].y;
        d[(32 + 2 * q) * 256 + tid] = prev[q].x; d[(32 + 2 * q + 1) * 256 + tid] = prev[q].y;
    }
#pragma unroll
    for (int i = 0; i < 16; ++i) u[i * 256 + tid] = kp.w[i];
}
template <int NP>
__device__ __forceinline__ void f32_state_load(const F32Args& A, int tid, float2 (&cur)[NP], float2 (&prev)[NP], KPackF& kp) {
    const float* d = reinterpret_cast<const float*>(reinterpret_cast<const char*>(A.skip_state) + (size_t)blockIdx.x * SHT_SKIP_STATE_BYTES_F32);
    const uint32_t* u = reinterpret_cast<const uint32_t*>(d + 64 * 256);
#pragma unroll
    for (int q = 0; q < NP; ++q) {
        cur[q] = make_float2(d[(2 * q) * 256 + tid], d[(2 * q + 1) * 256 + tid]);
        prev[q] = make_float2(d[(32 + 2 * q) * 256 + tid], d[(32 + 2 * q + 1) * 256 + tid]);
    }
#pragma unroll
    for (int i = 0; i < 16; ++i) kp.w[i] = u[i * 256 + tid];
}
// pairs this launch skips / runs: SM 0 transform (skip p0), 1 probe (all), 2 dump (the first p0 pairs only; false if there are none)
template <int SM>
__device__ __forceinline__ bool f32_skip_range(const F32Args& A, int mtop, int& m_first, int& m_last) {
    m_first = mtop; m_last = 0;
    if (SM == 1 || !A.skip_p0) return true;
    const int p0 = A.skip_p0[blockIdx.x];
    if (SM == 2) { m_last = mtop - 2 * p0 + 1; return p0 > 0; }
    m_first = mtop - 2 * p0;
    return true;
}


// =============================================================================================================
// inverse, Eq. 33:  F[row(+-m)][theta] += sum_l G[m][l][c] d^l_{m,0}(theta)
// warp w: degrees l0 + 8 w + j (j < 8); lane: ring pairs th0 + 2 lane + {0, 1} + 64 ip (ip < 2)
// =============================================================================================================
// FOLD (rings symmetric about the equator, northern half recursed): d^l_{m0}(pi - theta) = (-1)^{l+m} d^l_{m0}(theta).  The
// degrees of a warp all have one parity (warp w: l0 + 16 (w/2) + (w%2) + 2j), the reducers add the even-degree and the odd-degree warps
// apart (E0, E1) and write F_m(theta) = E0 + E1 and F_m(pi - theta) = (-1)^m (E0 - E1), as the fp64 kernel does.
template <int NC, bool FOLD, int SM>
__global__ void __launch_bounds__(NWF * 32, 2) theta_inverse_f32(const F32Args A) {
    constexpr int RL = 8, RP = 2, NP = RL * RP, DS = FOLD ? 2 : 1, C4 = 2 * NC;      // RP ring pairs per thread; C4 real columns
    __shared__ float4 s_ab[2][TLF];                  // {A, A, -B, -B} of the block's degrees: operands arrive duplicated for the packed math
    __shared__ float4 s_g[2][TLF * NC];              // {Re, Re, Im, Im} of G[m][l][c]
    __shared__ float s_lam[2][NTF];
    __shared__ float s_part[2][NWF][C4][NTF];        // planar partial sums, double-buffered: step m is reduced while step m-1 is computed
    const int ntt = A.ntp / NTF, nlt = A.Lp / TLF;
    const int lt = nlt - 1 - (int)(blockIdx.x / ntt), tt = blockIdx.x % ntt;      // heavy tiles first
    const int l0 = lt * TLF, th0 = tt * NTF;
    if (l0 >= A.L || th0 >= A.nth) return;
    const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
    const int mtop = min(l0 + TLF - 1, A.L - 1);
    int m_first, m_last;                              // steps m_first .. m_last of the recursion run in this launch (silent-head skip)
    if (!f32_skip_range<SM>(A, mtop, m_first, m_last)) return;
    bool contrib = false;                             // (probe) some item of this thread is in its last window
    const int la = FOLD ? l0 + 2 * RL * (w >> 1) + (w & 1) : l0 + w * RL;         // degrees of this warp: la + DS j

    // operand rows of step m, one element per thread, copied global -> shared asynchronously (cp.async): the copy of step m-1
    // is in flight while step m is computed and is awaited just before the block barrier.  The tables hold the duplicated form.
    auto load_ops = [&](int m, int buf) {
        if (tid < TLF) __pipeline_memcpy_async(&s_ab[buf][tid], &A.ab[(size_t)m * A.Lp + l0 + tid], sizeof(float4));
        if (tid < TLF * NC)
            __pipeline_memcpy_async(&s_g[buf][tid], reinterpret_cast<const float4*>(A.in) + ((size_t)m * A.Lp + l0) * NC + tid, sizeof(float4));
        if (tid >= 128 && tid < 128 + NTF)
            __pipeline_memcpy_async(&s_lam[buf][tid - 128], &A.lam32[(size_t)(m + 1) * A.ntp + th0 + tid - 128], sizeof(float));
        __pipeline_commit();
    };
    float2 cur[NP], prev[NP];
    KPackF kp;
    kp.fill(0u);
#pragma unroll
    for (int q = 0; q < NP; ++q) { cur[q] = make_float2(0.f, 0.f); prev[q] = make_float2(0.f, 0.f); }
    if (SM == 0 && m_first < mtop) f32_state_load<NP>(A, tid, cur, prev, kp);
    if (SM == 1 && tid == 0) A.skip_p0[blockIdx.x] = 1 << 30;
    load_ops(m_first, 0);
    __pipeline_wait_prior(0);
    __syncthreads();

    // cross-warp sum of the partial sums of step m (buffer pb) and RED.ADD to the output rows
    auto reduce = [&](const int m, const int pb) {
        for (int o = tid; o < NC * NTF; o += NWF * 32) {
            const int c = o / NTF, t = o % NTF, th = th0 + t;
            float ex = 0.f, ey = 0.f, ox = 0.f, oy = 0.f;
#pragma unroll
            for (int ww = 0; ww < NWF; ++ww) {
                const float vx = s_part[pb][ww][2 * c][t], vy = s_part[pb][ww][2 * c + 1][t];
                if (FOLD && (ww & 1)) { ox += vx; oy += vy; } else { ex += vx; ey += vy; }
            }
            if (th < A.nth && !(c == 1 && m == 0)) {
                const int m_out = c == 1 ? -m : m;
                const int row = m_out < 0 ? m_out + A.NB : m_out;
                double* op = reinterpret_cast<double*>(A.out) + ((size_t)row * A.ldout + th) * 2;
                red_add_f64(op, (double)(ex + ox)); red_add_f64(op + 1, (double)(ey + oy));
                const int tm = A.nfull - 1 - th;
                if (FOLD && tm != th) {
                    const float sg = (m & 1) ? -1.f : 1.f;
                    double* os = reinterpret_cast<double*>(A.out) + ((size_t)row * A.ldout + tm) * 2;
                    red_add_f64(os, (double)(sg * (ex - ox))); red_add_f64(os + 1, (double)(sg * (ey - oy)));
                }
            }
        }
    };
    // one step: project d_m, then advance to d_{m-1}.  `ca` holds d_m, `cb` holds d_{m+1} on entry and d_{m-1} on exit.
    auto step = [&](const int m, const int buf, float2 (&ca)[NP], float2 (&cb)[NP]) {
        if (m > 0) load_ops(m - 1, buf ^ 1);
        bool mine = m <= la + DS * (RL - 1) && la < A.L;   // this warp has started degrees
        if (mine && m >= la) {                      // the degree l == m starts (warp-uniform)
#pragma unroll
            for (int j = 0; j < RL; ++j)
                if (m == la + DS * j) {
#pragma unroll
                    for (int ip = 0; ip < RP; ++ip) {
                        const size_t o = (size_t)m * A.ntp + th0 + 2 * lane + 64 * ip;
                        ca[j * RP + ip] = *reinterpret_cast<const float2*>(A.st_val + o); cb[j * RP + ip] = make_float2(0.f, 0.f);
                        const ushort2 k2 = *reinterpret_cast<const ushort2*>(A.st_k + o);
                        kp.set(2 * (j * RP + ip), k2.x); kp.set(2 * (j * RP + ip) + 1, k2.y);
                        if (SM == 1 && (k2.x == 0 || k2.y == 0)) contrib = true;
                    }
                }
        }
        float2 acc[RP][C4];
#pragma unroll
        for (int ip = 0; ip < RP; ++ip)
#pragma unroll
            for (int c = 0; c < C4; ++c) acc[ip][c] = make_float2(0.f, 0.f);
        if (mine) {
            float2 lam[RP];
#pragma unroll
            for (int ip = 0; ip < RP; ++ip) lam[ip] = *reinterpret_cast<const float2*>(&s_lam[buf][2 * lane + 64 * ip]);
#pragma unroll
            for (int j = 0; j < RL; ++j) {
                const int dj = la - l0 + DS * j;
                const float4 ab = s_ab[buf][dj];
                const float2 A2 = make_float2(ab.x, ab.y), nB2 = make_float2(ab.z, ab.w);
                float2 cf[C4];
#pragma unroll
                for (int c = 0; c < NC; ++c) {
                    const float4 t = s_g[buf][dj * NC + c];
                    cf[2 * c] = make_float2(t.x, t.y); cf[2 * c + 1] = make_float2(t.z, t.w);
                }
#pragma unroll
                for (int ip = 0; ip < RP; ++ip) {
                    const float2 e = ca[j * RP + ip];
#pragma unroll
                    for (int c = 0; c < C4; ++c) acc[ip][c] = __ffma2_rn(e, cf[c], acc[ip][c]);
                    cb[j * RP + ip] = __ffma2_rn(__fmul2_rn(lam[ip], A2), e, __fmul2_rn(nB2, cb[j * RP + ip]));
                }
            }
            if (kp.any_nonzero()) window_check_f<NP, SM == 1>(cb, ca, kp, contrib);
        }
        const int pb = buf;                         // partial-sum buffer of this step (alternates with the operand buffer)
#pragma unroll
        for (int ip = 0; ip < RP; ++ip)
#pragma unroll
            for (int c = 0; c < C4; ++c) *reinterpret_cast<float2*>(&s_part[pb][w][c][2 * lane + 64 * ip]) = acc[ip][c];
        __pipeline_wait_prior(0);
        if (SM == 1) {                              // probe: first pair, 8 steps below the ramp or later, in which any thread contributes
            const int any = __syncthreads_or(f32_matters<NP>(cb, kp));
            if (tid == 0 && any && m < l0 - 8 && A.skip_p0[blockIdx.x] == (1 << 30)) A.skip_p0[blockIdx.x] = (mtop - m) / 2;
        } else
            __syncthreads();                        // the only block barrier of the step: partial sums of m and operands of m-1 are visible;
        reduce(m, pb);                              // buffer pb is next written two steps from now, after the barrier of step m-1
    };
    for (int m = m_first; m >= m_last; m -= 2) {
        step(m, (m_first - m) & 1, cur, prev);
        if (m - 1 >= m_last) step(m - 1, (m_first - m + 1) & 1, prev, cur);
    }
    if (SM == 2) f32_state_store<NP>(A, tid, cur, prev, kp);
}

// =============================================================================================================
// forward, Eq. 30:  H[+-m + L-1][l] += sum_theta W[m][theta][c] d^l_{m,0}(theta)
// warp w: ring pairs th0 + 16 w + 2 ip + {0, 1} (ip < 8); lane: degrees l0 + lane + 32 r (r < 2)
// FOLD: northern rings only; W32 rows hold E = q (F_m(theta) + F_m(pi - theta)) and O = q (F_m(theta) - F_m(pi - theta)); a degree
// with l+m even contracts with E, one with l+m odd with O (d^l_{m0}(pi - theta) = (-1)^{l+m} d^l_{m0}(theta)).  A thread's two
// degrees share their parity, which alternates with the lane: one load with two addresses serves both (as in theta_kernels.cu).
// =============================================================================================================
template <int NC, bool FOLD, int SM>
__global__ void __launch_bounds__(NWF * 32, 2) theta_forward_f32(const F32Args A) {
    constexpr int RL = 2, RP = 8, NP = RL * RP, NSET = FOLD ? 2 : 1, C4 = 2 * NC, NPB = NTF / 2;      // NPB ring pairs per block
    __shared__ float4 s_ab[2][TLF];
    __shared__ __align__(16) float2 s_w[2][NPB * NSET * C4];      // [pair][set][column] = (ring 2p, ring 2p+1): the layout of k_weight_split_f32
    __shared__ float s_lam[2][NTF];
    __shared__ float s_part[2][NWF][C4][TLF];
    const int ntt = A.ntp / NTF, nlt = A.Lp / TLF;
    const int lt = nlt - 1 - (int)(blockIdx.x / ntt), tt = blockIdx.x % ntt;
    const int l0 = lt * TLF, th0 = tt * NTF;
    if (l0 >= A.L || th0 >= A.nth) return;
    const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
    const int mtop = min(l0 + TLF - 1, A.L - 1);
    int m_first, m_last;
    if (!f32_skip_range<SM>(A, mtop, m_first, m_last)) return;
    bool contrib = false;

    auto load_ops = [&](int m, int buf) {
        if (tid < TLF) __pipeline_memcpy_async(&s_ab[buf][tid], &A.ab[(size_t)m * A.Lp + l0 + tid], sizeof(float4));
        const float4* src = reinterpret_cast<const float4*>(A.in + ((size_t)m * A.ntp + th0) * NSET * NC);
        for (int o = tid; o < NPB * NSET * C4 / 2; o += NWF * 32)
            __pipeline_memcpy_async(reinterpret_cast<float4*>(&s_w[buf][0]) + o, src + o, sizeof(float4));
        if (tid >= 128 && tid < 128 + NTF)
            __pipeline_memcpy_async(&s_lam[buf][tid - 128], &A.lam32[(size_t)(m + 1) * A.ntp + th0 + tid - 128], sizeof(float));
        __pipeline_commit();
    };
    float2 cur[NP], prev[NP];
    KPackF kp;
    kp.fill(0u);
#pragma unroll
    for (int q = 0; q < NP; ++q) { cur[q] = make_float2(0.f, 0.f); prev[q] = make_float2(0.f, 0.f); }
    int lr[RL];
#pragma unroll
    for (int r = 0; r < RL; ++r) lr[r] = l0 + lane + 32 * r;
    if (SM == 0 && m_first < mtop) f32_state_load<NP>(A, tid, cur, prev, kp);
    if (SM == 1 && tid == 0) A.skip_p0[blockIdx.x] = 1 << 30;
    load_ops(m_first, 0);
    __pipeline_wait_prior(0);
    __syncthreads();

    auto step = [&](const int m, const int buf, float2 (&ca)[NP], float2 (&cb)[NP]) {
        if (m > 0) load_ops(m - 1, buf ^ 1);
#pragma unroll
        for (int r = 0; r < RL; ++r)
            if (m == lr[r] && lr[r] < A.L) {        // this lane's degree starts
#pragma unroll
                for (int ip = 0; ip < RP; ++ip) {
                    const size_t o = (size_t)m * A.ntp + th0 + w * 2 * RP + 2 * ip;
                    ca[r * RP + ip] = *reinterpret_cast<const float2*>(A.st_val + o); cb[r * RP + ip] = make_float2(0.f, 0.f);
                    const ushort2 k2 = *reinterpret_cast<const ushort2*>(A.st_k + o);
                    kp.set(2 * (r * RP + ip), k2.x); kp.set(2 * (r * RP + ip) + 1, k2.y);
                    if (SM == 1 && (k2.x == 0 || k2.y == 0)) contrib = true;
                }
            }
        float2 acc[RL][C4];
#pragma unroll
        for (int r = 0; r < RL; ++r)
#pragma unroll
            for (int c = 0; c < C4; ++c) acc[r][c] = make_float2(0.f, 0.f);
        float2 A2[RL], nB2[RL];
#pragma unroll
        for (int r = 0; r < RL; ++r) { const float4 ab = s_ab[buf][lane + 32 * r]; A2[r] = make_float2(ab.x, ab.y); nB2[r] = make_float2(ab.z, ab.w); }
        const int set = FOLD ? ((l0 + m + lane) & 1) : 0;      // FOLD: 0 = E (l+m even), 1 = O; per lane parity, same for both degrees
        const float2* wrow = &s_w[buf][(w * RP * NSET + set) * C4];
        const float2* lrow = reinterpret_cast<const float2*>(&s_lam[buf][w * 2 * RP]);
#pragma unroll
        for (int ip = 0; ip < RP; ++ip) {
            const float2 lam = lrow[ip];
            float2 wv[C4];
#pragma unroll
            for (int c = 0; c < NC; ++c) {
                const float4 t = *reinterpret_cast<const float4*>(wrow + ip * NSET * C4 + 2 * c);
                wv[2 * c] = make_float2(t.x, t.y); wv[2 * c + 1] = make_float2(t.z, t.w);
            }
#pragma unroll
            for (int r = 0; r < RL; ++r) {
                const float2 e = ca[r * RP + ip];
#pragma unroll
                for (int c = 0; c < C4; ++c) acc[r][c] = __ffma2_rn(e, wv[c], acc[r][c]);
                cb[r * RP + ip] = __ffma2_rn(__fmul2_rn(lam, A2[r]), e, __fmul2_rn(nB2[r], cb[r * RP + ip]));
            }
        }
        if (kp.any_nonzero()) window_check_f<NP, SM == 1>(cb, ca, kp, contrib);
#pragma unroll
        for (int r = 0; r < RL; ++r)
#pragma unroll
            for (int c = 0; c < C4; ++c) s_part[buf][w][c][lane + 32 * r] = acc[r][c].x + acc[r][c].y;      // the pair's two rings
        __pipeline_wait_prior(0);
        if (SM == 1) {
            const int any = __syncthreads_or(f32_matters<NP>(cb, kp));
            if (tid == 0 && any && m < l0 - 8 && A.skip_p0[blockIdx.x] == (1 << 30)) A.skip_p0[blockIdx.x] = (mtop - m) / 2;
        } else
            __syncthreads();                        // the only block barrier of the step (partial sums double-buffered, see the inverse)
        for (int o = tid; o < NC * TLF; o += NWF * 32) {
            const int c = o / TLF, t = o % TLF, l = l0 + t;
            float sx = 0.f, sy = 0.f;
#pragma unroll
            for (int ww = 0; ww < NWF; ++ww) { sx += s_part[buf][ww][2 * c][t]; sy += s_part[buf][ww][2 * c + 1][t]; }
            if (l < A.L && l >= m && !(c == 1 && m == 0)) {
                const int m_out = c == 1 ? -m : m;
                double* op = reinterpret_cast<double*>(A.out) + ((size_t)(m_out + A.L - 1) * A.Lp + l) * 2;
                red_add_f64(op, (double)sx); red_add_f64(op + 1, (double)sy);
            }
        }
    };
    for (int m = m_first; m >= m_last; m -= 2) {
        step(m, (m_first - m) & 1, cur, prev);
        if (m - 1 >= m_last) step(m - 1, (m_first - m + 1) & 1, prev, cur);
    }
    if (SM == 2) f32_state_store<NP>(A, tid, cur, prev, kp);
}

}  // namespace

template <int SM>
static void launch_f32_mode(const F32Args& a, bool forward, int NC, dim3 grid, cudaStream_t st) {
    if (forward && a.fold0) {
        if (NC == 2) theta_forward_f32<2, true, SM><<<grid, NWF * 32, 0, st>>>(a);
        else theta_forward_f32<1, true, SM><<<grid, NWF * 32, 0, st>>>(a);
    } else if (forward) {
        if (NC == 2) theta_forward_f32<2, false, SM><<<grid, NWF * 32, 0, st>>>(a);
        else theta_forward_f32<1, false, SM><<<grid, NWF * 32, 0, st>>>(a);
    } else if (a.fold0) {
        if (NC == 2) theta_inverse_f32<2, true, SM><<<grid, NWF * 32, 0, st>>>(a);
        else theta_inverse_f32<1, true, SM><<<grid, NWF * 32, 0, st>>>(a);
    } else {
        if (NC == 2) theta_inverse_f32<2, false, SM><<<grid, NWF * 32, 0, st>>>(a);
        else theta_inverse_f32<1, false, SM><<<grid, NWF * 32, 0, st>>>(a);
    }
}
cudaError_t launch_theta_f32(const F32Args& a, bool forward, int NC, cudaStream_t st) {
    dim3 grid((a.Lp / TLF) * (a.ntp / NTF));
    if (a.skip_mode == 1) launch_f32_mode<1>(a, forward, NC, grid, st);
    else if (a.skip_mode == 2) launch_f32_mode<2>(a, forward, NC, grid, st);
    else launch_f32_mode<0>(a, forward, NC, grid, st);
    count_launch();
    return cudaGetLastError();
}
