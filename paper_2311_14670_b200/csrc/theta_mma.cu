// theta_mma.cu -- the batched hot path (BASELINE config 5b): one Wigner-d recursion (Eq. 25-27,
// PAPER.md:225-234) shared by a batch of maps.  With B maps the theta / l contraction of Eq. 30 / Eq. 33
// is a dense GEMM per harmonic order m,
//     inverse  F_m[theta][col] = sum_l     e^l_m(theta) * G_m[l][col]
//     forward  H_m[l][col]     = sum_theta e^l_m(theta) * W_m[theta][col],        col = (map, +-m, re/im),
// whose left operand e^l_m(theta) is never stored: it is produced in registers by the recursion and fed straight into
// FP64 tensor-core MMAs (mma.sync m8n8k4, SASS DMMA.8x8x4; tcgen05 has no FP64 kind).
//
// Mapping.  DMMA computes D(8x8) += A(8x4) B(4x8); lane (gid = lane/4, tig = lane%4) holds A[gid][tig], B[tig][gid],
// D[gid][2 tig + {0,1}].  The contraction index K (degrees on the inverse, rings on the forward) runs over tig, the
// output row index M (rings on the inverse, degrees on the forward) over gid.  A thread carries NJ x NIB = 16 x 2
// recursion items (K = 4 jb + tig, M = 8 ib + gid): every iterate register IS an A fragment.  A warp therefore owns
// 64 K-values x 16 M-rows and needs no cross-warp reduction; the CTA (8 compute warps) owns 64 K x 128 M.  Per
// recursion step a warp issues 128 DMMA (16 jb x 2 ib x 4 column tiles of 8 = 32 real columns) and 64 DMUL/DFMA of
// recursion; B fragments come from a TMA-filled shared-memory ring (rows padded to 36 doubles: conflict-free LDS.64).
// The warp's 16 x 32 result tile goes to a private staging buffer and is added to global memory by ONE bulk-reduce
// TMA (cp.reduce.async.bulk .add.f64) -- no per-element RED, no reducer warps.
// Renormalisation windows, peak split and dead-ring handling are those of theta_kernels.cu (internal.h).
#include "device_utils.cuh"
#include "internal.h"

#include <cuda_runtime.h>
#include <stdint.h>

namespace {

using namespace shtdev;

__device__ __forceinline__ void dmma(double (&c)[2], double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                 : "+d"(c[0]), "+d"(c[1])
                 : "d"(a), "d"(b));
}
constexpr int NW = 8;        // compute warps
constexpr int NAUX = 4;      // auxiliary warpgroup (one thread of it is the TMA producer)
constexpr int NJ = 16;       // K blocks of 4 per thread
constexpr int NIB = 2;       // M blocks of 8 per thread
constexpr int NI = NJ * NIB; // recursion items per thread
constexpr int NT8 = SHT_MMA_NCOL / 8;
constexpr int ROW = SHT_MMA_ROW;
constexpr int TK = 4 * NJ;          // 64: contraction extent of a CTA
constexpr int TM = NW * 8 * NIB;    // 128: output rows of a CTA
constexpr int NSTG = 4;             // operand ring stages
static_assert(TK == SHT_TQ, "the contraction tile is one kappa quantum");

using KPack32 = KPack<NI>;

// FOLD (forward, n = 0, northern rings only): an operand row holds two column sets, E = q (F_m(theta) + F_m(pi - theta)) and
// O = q (F_m(theta) - F_m(pi - theta)); a degree with l+m even contracts with E, one with l+m odd with O (PAPER.md:236,
// d^l_{m0}(pi - theta) = (-1)^{l+m} d^l_{m0}(theta)).  The M rows of one DMMA are then the 8 degrees mw0 + 2 gid + ib of equal parity.
template <int ROW_>
struct MmaSmem {
    double op[NSTG][TK * ROW_];     // operand rows of the CTA's 64 K-values: 32 columns + side columns (TMA ring)
    double side[NSTG][TM];          // inverse: lambda_m(theta) of the CTA's 128 rings; forward: (s, G) of its 2 quanta
    double stg[NW][2][16 * SHT_MMA_NCOL];   // per-warp result tiles (double-buffered source of the bulk reduce)
    uint64_t full[NSTG], empty[NSTG];
};

// FWD = false: inverse (K = degrees, M = rings).  FWD = true: forward (K = rings, M = degrees).
template <bool FWD, bool FOLD>
__global__ void __launch_bounds__((NW + NAUX) * 32, 1) theta_mma_kernel(const MmaArgs A) {
    static_assert(FWD || !FOLD, "the fold is a forward variant");
    constexpr int ROW = FOLD ? SHT_MMA_ROWF : SHT_MMA_ROW;       // shadows the namespace constant
    constexpr int SIDE = FOLD ? 2 * SHT_MMA_NCOL : SHT_MMA_NCOL;  // index of the first side column of an operand row
    extern __shared__ __align__(128) unsigned char smem_raw[];
    MmaSmem<ROW>& sm = *reinterpret_cast<MmaSmem<ROW>*>(smem_raw);

    const ThetaPass P = A.passes[blockIdx.y];
    const int cg = blockIdx.z;
    // degree tiles: TK (inverse) / TM (forward) degrees; ring tiles: TM (inverse) / TK (forward) rings
    constexpr int TLD = FWD ? TM : TK, TTH = FWD ? TK : TM;
    const int ntt = A.ntp / TTH, nlt = A.Lp / TLD;
    const int lt = nlt - 1 - (int)(blockIdx.x / ntt), tt = blockIdx.x % ntt;      // heavy (large-l) tiles first
    const int l0 = lt * TLD, th0 = tt * TTH;
    const int an = P.n < 0 ? -P.n : P.n;
    if (l0 + TLD <= an || l0 >= A.L || th0 >= A.nth) return;
    const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
    const int mtop = min(l0 + TLD - 1, A.L - 1), m_end = P.m_end;
    const int nsteps = mtop - m_end + 1;
    const int Mp = FWD ? A.Lp : A.ntp, Kp = FWD ? A.ntp : A.Lp;     // padded extents of the M and K axes
    const int k0 = FWD ? th0 : l0, m0 = FWD ? l0 : th0;

    if (tid == 0) {
        for (int i = 0; i < NSTG; ++i) { mbar_init(&sm.full[i], 1); mbar_init(&sm.empty[i], NW); }
        mbar_fence_init();
    }
    __syncthreads();

    if (w >= NW) {
        // ------------------------------------------------------------------------- TMA producer (one thread)
        reg_dealloc_aux();
        if (tid != NW * 32) return;
        const double* in = P.in + (size_t)cg * A.in_cg_stride;
        constexpr uint32_t op_bytes = TK * ROW * sizeof(double);
        for (int it = 0; it < nsteps; ++it) {
            const int m = mtop - it, slot = it & (NSTG - 1);
            if (it >= NSTG) mbar_wait(&sm.empty[slot], ((it / NSTG) & 1) ^ 1);
            const size_t row = (size_t)(m - m_end);
            if (FWD) {
                mbar_expect_tx(&sm.full[slot], op_bytes + 2 * (uint32_t)sizeof(double2));
                bulk_g2s(&sm.op[slot][0], in + (row * Kp + k0) * ROW, op_bytes, &sm.full[slot]);
                const double2* sg = A.sg + (size_t)(l0 / SHT_TQ) * A.sgstride + (m - A.mmin);
                bulk_g2s(&sm.side[slot][0], sg, sizeof(double2), &sm.full[slot]);
                bulk_g2s(&sm.side[slot][2], sg + A.sgstride, sizeof(double2), &sm.full[slot]);
            } else {
                mbar_expect_tx(&sm.full[slot], op_bytes + TM * (uint32_t)sizeof(double));
                bulk_g2s(&sm.op[slot][0], in + (row * Kp + k0) * ROW, op_bytes, &sm.full[slot]);
                bulk_g2s(&sm.side[slot][0], P.lam + (row + 1) * A.ntp + th0, TM * sizeof(double), &sm.full[slot]);
            }
        }
        return;
    }
    reg_alloc_compute();

    // ----------------------------------------------------------------------------- compute warps
    const int gid = lane >> 2, tig = lane & 3;
    const int mw0 = m0 + w * 8 * NIB;                   // first M row of this warp
    auto mrow = [&](int ib) { return FOLD ? 2 * gid + ib : 8 * ib + gid; };   // M row (within the warp's 16) of the thread's block ib
    // forward: this warp's degrees are mw0 .. mw0+15 (inside one quantum); inverse: the CTA's 64 degrees are shared
    const int l_hi = FWD ? mw0 + 8 * NIB - 1 : l0 + TK - 1;       // highest degree this warp touches
    const int l_lo = FWD ? mw0 : l0;
    const bool warp_real = l_lo < A.L;
    double cur[NI], prev[NI];
    KPack32 kp;
    kp.fill(0xffffffffu);
#pragma unroll
    for (int q = 0; q < NI; ++q) { cur[q] = 0.0; prev[q] = 0.0; }
    bool wact = false;
    int mlo[NIB];
    double lr[NIB];                                     // forward: degree of the thread's M rows (as double)
#pragma unroll
    for (int ib = 0; ib < NIB; ++ib) {
        const int mi = mw0 + mrow(ib);
        mlo[ib] = -(1 << 30);
        if (!FWD) {
            if (P.m_lo) mlo[ib] = P.m_lo[mi];
            if (mi >= A.nth) mlo[ib] = 1 << 30;          // padded rings never contribute
        }
        lr[ib] = (double)mi;
    }
    double* const out = reinterpret_cast<double*>(P.out) + (size_t)cg * A.out_cg_stride + (size_t)mw0 * SHT_MMA_NCOL;
    int obuf = 0;

    // one recursion step; `ca` holds e_m, `cb` holds e_{m+1} on entry and e_{m-1} on exit (roles swap every step)
    auto step = [&](const int m, const int slot, double (&ca)[NI], double (&cb)[NI]) {
        const double* op = &sm.op[slot][0];
        // ---- Eq. 27 start values of the degree l == m (items of that degree were all-zero so far)
        if (m >= l_lo) {
            if (FWD) {
                const int d = m - mw0, ibs = FOLD ? (d & 1) : (d >> 3);
                if (gid == (FOLD ? (d >> 1) : (d & 7))) {
                    const double* sv = P.st_val + (size_t)m * A.ntp + th0 + tig;
                    const uint8_t* sk = P.st_k + (size_t)m * A.ntp + th0 + tig;
#pragma unroll
                    for (int ib = 0; ib < NIB; ++ib)
                        if (ib == ibs) {
#pragma unroll
                            for (int jb = 0; jb < NJ; ++jb) {
                                ca[jb * NIB + ib] = sv[4 * jb]; cb[jb * NIB + ib] = 0.0;
                                kp.set(jb * NIB + ib, sk[4 * jb]);
                            }
                        }
                }
            } else {
                const int d = m - l0, jbs = d >> 2;
                if (tig == (d & 3)) {
                    const double* sv = P.st_val + (size_t)m * A.ntp + mw0 + gid;
                    const uint8_t* sk = P.st_k + (size_t)m * A.ntp + mw0 + gid;
#pragma unroll
                    for (int jb = 0; jb < NJ; ++jb)
                        if (jb == jbs) {
#pragma unroll
                            for (int ib = 0; ib < NIB; ++ib) {
                                ca[jb * NIB + ib] = sv[8 * ib]; cb[jb * NIB + ib] = 0.0;
                                kp.set(jb * NIB + ib, sk[8 * ib]);
                            }
                        }
                }
            }
            wact = true;                                // re-evaluated at the next window check
        }
        // ---- recursion coefficients: lambda'_m = lambda_m s_m along the ring axis, g'_m = (l-m)(l+m+1) G_m along the degree axis
        double cM[NIB];                                 // the coefficient that depends on the M row
        double sK;                                      // scale applied to the K-dependent side column
        if (FWD) {
            const double2 sg = *reinterpret_cast<const double2*>(&sm.side[slot][2 * (w >> 2)]);
            sK = sg.x;
            const double dm = (double)m;
#pragma unroll
            for (int ib = 0; ib < NIB; ++ib) cM[ib] = (lr[ib] - dm) * (lr[ib] + dm + 1.0) * sg.y;
        } else {
            const double s = op[ROW - 3];               // column 33 of row 0: s_m of the CTA's quantum
            sK = 1.0;
#pragma unroll
            for (int ib = 0; ib < NIB; ++ib) cM[ib] = sm.side[slot][w * 8 * NIB + 8 * ib + gid] * s;
        }
        const double* kr = op + tig * ROW;              // row of K = 4 jb + tig is kr + 4 jb ROW
        const int par0 = (mw0 + m) & 1;                 // FOLD: parity of l + m of block ib = 0 (block 1 has the other one)
        if (wact) {
            double acc[NIB][NT8][2];
#pragma unroll
            for (int ib = 0; ib < NIB; ++ib)
#pragma unroll
                for (int nt = 0; nt < NT8; ++nt) { acc[ib][nt][0] = 0.0; acc[ib][nt][1] = 0.0; }
#pragma unroll
            for (int jb = 0; jb < NJ; ++jb) {
                const double* r = kr + 4 * jb * ROW;
                double b[FOLD ? NIB : 1][NT8];            // FOLD: block ib contracts with the column set of its parity
#pragma unroll
                for (int s2 = 0; s2 < (FOLD ? NIB : 1); ++s2)
#pragma unroll
                    for (int nt = 0; nt < NT8; ++nt) b[s2][nt] = r[(FOLD ? ((par0 ^ s2) & 1) * SHT_MMA_NCOL : 0) + 8 * nt + gid];
                const double cK = r[SIDE] * sK;           // inverse: g'_m(l); forward: lambda_m(theta) s_m
#pragma unroll
                for (int ib = 0; ib < NIB; ++ib) {
                    const double e = ca[jb * NIB + ib];
#pragma unroll
                    for (int nt = 0; nt < NT8; ++nt) dmma(acc[ib][nt], e, b[FOLD ? ib : 0][nt]);
                    if (FWD) cb[jb * NIB + ib] = fma(cK, e, -(cM[ib] * cb[jb * NIB + ib]));
                    else cb[jb * NIB + ib] = fma(cM[ib], e, -(cK * cb[jb * NIB + ib]));
                }
            }
            __syncwarp();
            if (lane == 0) { mbar_arrive(&sm.empty[slot]); bulk_wait_read<1>(); }    // the buffer used two tiles ago is free
            __syncwarp();
            double* sb = &sm.stg[w][obuf][0];
#pragma unroll
            for (int ib = 0; ib < NIB; ++ib) {
                const bool keep = m >= mlo[ib];
#pragma unroll
                for (int nt = 0; nt < NT8; ++nt)
                    *reinterpret_cast<double2*>(sb + mrow(ib) * SHT_MMA_NCOL + 8 * nt + 2 * tig) =
                        keep ? make_double2(acc[ib][nt][0], acc[ib][nt][1]) : make_double2(0.0, 0.0);
            }
            fence_async_smem();
            __syncwarp();
            if (lane == 0) {
                bulk_reduce_add_f64(out + (size_t)(m - m_end) * Mp * SHT_MMA_NCOL, sb, 16 * SHT_MMA_NCOL * sizeof(double));
                bulk_commit();
            }
            obuf ^= 1;
        } else {                                        // every item of the warp is still below 2^-340: recursion only
#pragma unroll
            for (int jb = 0; jb < NJ; ++jb) {
                const double cK = kr[4 * jb * ROW + SIDE] * sK;
#pragma unroll
                for (int ib = 0; ib < NIB; ++ib) {
                    if (FWD) cb[jb * NIB + ib] = fma(cK, ca[jb * NIB + ib], -(cM[ib] * cb[jb * NIB + ib]));
                    else cb[jb * NIB + ib] = fma(cM[ib], ca[jb * NIB + ib], -(cK * cb[jb * NIB + ib]));
                }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(&sm.empty[slot]);
        }
        if ((m & (SHT_JCHK - 1)) == 0) {
            if (kp.any_nonzero()) {
                const double s = pow2i(-SHT_SWIN);
#pragma unroll
                for (int q = 0; q < NI; ++q)
                    if (hi_abs(cb[q]) > SHT_HI_TWIN && kp.get(q) != 0u && kp.get(q) != 0xffu) { cb[q] *= s; ca[q] *= s; kp.dec(q); }
            }
            if (P.m_lo) {
#pragma unroll
                for (int q = 0; q < NI; ++q)
                    if (hi_abs(cb[q]) > SHT_HI_DEAD) { cb[q] = 0.0; ca[q] = 0.0; }
            }
            if (m < l_lo) wact = __any_sync(0xffffffffu, kp.any_zero_byte());
        }
    };

    for (int it = 0; it < nsteps; it += 2) {
        {
            const int slot = it & (NSTG - 1);
            mbar_wait(&sm.full[slot], (it / NSTG) & 1);
            const int m = mtop - it;
            if (m <= l_hi && warp_real) step(m, slot, cur, prev);
            else { __syncwarp(); if (lane == 0) mbar_arrive(&sm.empty[slot]); }
        }
        if (it + 1 < nsteps) {
            const int slot = (it + 1) & (NSTG - 1);
            mbar_wait(&sm.full[slot], ((it + 1) / NSTG) & 1);
            const int m = mtop - it - 1;
            if (m <= l_hi && warp_real) step(m, slot, prev, cur);
            else { __syncwarp(); if (lane == 0) mbar_arrive(&sm.empty[slot]); }
        }
    }
    if (lane == 0) bulk_wait_read<0>();                 // shared memory must outlive the last bulk reduce's reads
}

}  // namespace

template <bool FWD, bool FOLD>
static cudaError_t launch_mma(const MmaArgs& a, cudaStream_t st) {
    const size_t smem = sizeof(MmaSmem<FOLD ? SHT_MMA_ROWF : SHT_MMA_ROW>) + 128;
    cudaError_t e = cudaFuncSetAttribute(theta_mma_kernel<FWD, FOLD>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    dim3 grid(FWD ? (a.Lp / TM) * (a.ntp / TK) : (a.Lp / TK) * (a.ntp / TM), a.npass, a.ncg);
    theta_mma_kernel<FWD, FOLD><<<grid, (NW + NAUX) * 32, smem, st>>>(a);
    count_launch();
    return cudaGetLastError();
}

cudaError_t launch_theta_mma(const MmaArgs& a, bool forward, cudaStream_t st) {
    if (a.npass == 0) return cudaSuccess;
    if (!forward) return launch_mma<false, false>(a, st);
    return a.fold0 ? launch_mma<true, true>(a, st) : launch_mma<true, false>(a, st);
}
