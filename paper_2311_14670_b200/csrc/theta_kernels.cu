// theta_kernels.cu -- the hot path: Wigner-d recursion in m (Eq. 25-27) fused with the theta
// contraction of Eq. 30 (forward, sum over rings) and Eq. 33 (inverse, sum over l) -- "interleaving recursion and
// computation", Sec. 4.4.  d-values live only in registers; nothing O(L^3) touches memory.
//
// Structure.  One CTA per SM: NW = 8 compute warps + 4 auxiliary warps (register budgets re-split
// with setmaxnreg: 232 / 40 per thread), no block-wide barrier in the m-loop.
//   compute warps: every thread carries an RL x RT register tile of (l, ring) items, 32 items, and per recursion
//       step does 1 DMUL + 1 DFMA (recursion, internal.h) and 2 (one order) or 4 (+-m) DFMA (projection) per item.
//       Operands that are uniform across the warp are shared-memory broadcasts.
//       inverse: lane <-> ring, registers <-> RL degrees x RT rings;  sum_l = in-thread FMA chains over RL degrees
//       forward: lane <-> degree, registers <-> RL degrees x RT rings; sum_theta = in-thread FMA chains over RT rings
//   auxiliary warp: (1) streams the per-step operand rows into a 4-stage ring with 1-D TMA bulk copies
//       (cp.async.bulk + mbarrier complete_tx), (2) forward only: scales the lambda row by the step's power of two,
//       (3) adds the per-warp partial sums of every step and issues RED.ADD.F64 to the output rows.
//   compute <-> auxiliary hand-off is a two-stage mbarrier pipeline (rfull / rempty); operand slots are recycled by the
//       auxiliary warp right after the reduction of the step that used them.
// All (l,m)-only and (theta,m)-only factors arrive as O(L^2) tables prepared by staging.cu.
#include "device_utils.cuh"
#include "internal.h"

#include <cuda_runtime.h>
#include <stdint.h>

namespace {

using namespace shtdev;

constexpr int NST = 4;   // stages of the operand ring
constexpr int NRS = 4;   // stages of the partial-sum hand-off of the forward kernel (131 KB; 2 -> 4: config 2 forward 0.814 -> 0.796 ms, L = 4096 19.34 -> 19.23 ms;
                         // starting half of the compute warps half a pair late, so that the two warps of a scheduler interleave, LOSES 7 % at either depth)
constexpr int KS = 2;    // recursion steps per pipeline stage (one TMA barrier, one hand-off per KS steps)
constexpr int NAUX = 4;  // auxiliary warps (one warpgroup: setmaxnreg works on aligned groups of 4 warps)

// ---- skipping the silent head of a tile (internal.h, ThetaArgs::skip_*) ------------------------------------------------------------
// [pbeg, pend): the pairs this launch runs for the block `bid`; returns false if the block has nothing to do in this mode
template <int SM>
__device__ __forceinline__ bool skip_range(const ThetaArgs& A, unsigned bid, int npairs, int& pbeg, int& pend) {
    pbeg = 0; pend = npairs;
    if (SM == 1 || !A.skip_p0) return true;                   // probe: the whole recursion
    const int p0 = A.skip_p0[bid];
    if (SM == 2) { pend = p0; return p0 > 0; }                // dump: the silent head only
    pbeg = p0;                                                // transform: start where the head ends
    return true;
}
// probe: does any item of the warp matter yet?  An iterate contributes to the sums through c_m(l) e (internal.h), c <= 2^250; one whose
// last window is reached (k = 0) but whose magnitude is still below 2^-330 adds less than 2^-80 of an O(1) sum: as silent as one with k > 0.
#define SHT_HI_SIGNIF ((1023 - 330) << 20)
template <int NI>
__device__ __forceinline__ bool warp_matters(const double (&cur)[NI], const KPack<NI>& kp) {
    bool big = false;
#pragma unroll
    for (int q = 0; q < NI; ++q) big = big || (kp.get(q) == 0u && hi_abs(cur[q]) > SHT_HI_SIGNIF);
    return __any_sync(0xffffffffu, big);
}
template <int NI>
__device__ __forceinline__ void skip_store(const ThetaArgs& A, unsigned bid, int ctid, const double (&cur)[NI], const double (&prev)[NI],
                                           const KPack<NI>& kp, bool wact) {
    static_assert(NI <= 32, "state layout: room for 32 items per thread");
    double* d = reinterpret_cast<double*>(reinterpret_cast<char*>(A.skip_state) + (size_t)bid * SHT_SKIP_STATE_BYTES);
    uint32_t* u = reinterpret_cast<uint32_t*>(d + 64 * 256);
#pragma unroll
    for (int q = 0; q < NI; ++q) { d[q * 256 + ctid] = cur[q]; d[(NI + q) * 256 + ctid] = prev[q]; }
#pragma unroll
    for (int i = 0; i < (NI + 3) / 4; ++i) u[i * 256 + ctid] = kp.w[i];
    u[8 * 256 + ctid] = wact ? 1u : 0u;
}
template <int NI>
__device__ __forceinline__ void skip_load(const ThetaArgs& A, unsigned bid, int ctid, double (&cur)[NI], double (&prev)[NI], KPack<NI>& kp, bool& wact) {
    const double* d = reinterpret_cast<const double*>(reinterpret_cast<const char*>(A.skip_state) + (size_t)bid * SHT_SKIP_STATE_BYTES);
    const uint32_t* u = reinterpret_cast<const uint32_t*>(d + 64 * 256);
#pragma unroll
    for (int q = 0; q < NI; ++q) { cur[q] = d[q * 256 + ctid]; prev[q] = d[(NI + q) * 256 + ctid]; }
#pragma unroll
    for (int i = 0; i < (NI + 3) / 4; ++i) kp.w[i] = u[i * 256 + ctid];
    wact = u[8 * 256 + ctid] != 0u;
}

// =============================================================================================================
// inverse theta step, Eq. 33:  F[row(m_out)][theta] += sum_l G[m][l] * e^l_m(theta)      (G carries c_m(l))
// block tile: TL = NW*RL degrees x NTH = 32*RT rings; KS = 2 recursion steps per pipeline stage
// =============================================================================================================
// FOLD (n = 0 on a ring set symmetric about the equator): only the northern rings are recursed.  d^l_{m0}(pi - theta) =
// (-1)^{l+m} d^l_{m0}(theta), so with E = sum over l+m even and O = sum over l+m odd of G d:
// F_m(theta) = E + O and F_m(pi - theta) = E - O.  The degrees of a WARP all have one parity (warp w: degrees
// l0 + 16 (w/2) + (w%2) + 2j), so every warp still hands over ONE partial-sum set -- the shared-memory footprint of the plain kernel,
// 128-ring tiles included -- and the reducers add the even-degree warps and the odd-degree warps apart and emit both rings.
// WT = ring groups of warps: the NW compute warps form ND = NW / WT degree groups x WT ring groups; a warp covers RL degrees x 32 RT rings.
// WT = 2 (16 degrees x 64 rings per warp) halves the cross-warp sum: half the partial-sum stores, half the reducers' loads and adds, and a
// hand-off twice as deep in the same shared memory, for twice the (broadcast) operand loads per item.
template <int RL, int RT, int NW, int NC, bool FOLD, int WT>
struct InvSmem {
    static constexpr int ND = NW / WT, TL = ND * RL, NTH = 32 * RT * WT, ROWD = 2 * NC + 2, NSET = FOLD ? 2 : 1;   // NSET: sets the reducers keep apart
    static constexpr int NRS = (NC == 1 || WT >= 2) ? 4 : 2;   // smaller partial-sum sets: a deeper hand-off fits
    double op[NST][KS][TL * ROWD];          // operand rows {c Re, c Im (x NC), g', s} of the block's degrees (TMA ring)
    double lam[NST][KS][NTH];               // lambda_m(theta) of the block's rings (TMA ring)
    double red[NRS][KS][ND][NTH][2 * NC];   // partial sums per degree group (the WT warps of a group own disjoint rings)
    int act[NRS][NW];                       // bit h: the warp wrote partial sums for step h of the pair
    uint64_t full[NST], rfull[NRS], rempty[NRS];
};

// SM: 0 = transform, 1 = probe, 2 = dump (ThetaArgs::skip_mode; separate instantiations keep the transform kernels free of the plan-time code)
template <int RL, int RT, int NW, int NC, bool FOLD, int WT, int SM>
__global__ void __launch_bounds__((NW + NAUX) * 32, 1) theta_inverse_kernel(const ThetaArgs A) {
    using S = InvSmem<RL, RT, NW, NC, FOLD, WT>;
    constexpr int TL = S::TL, NTH = S::NTH, NI = RL * RT, ROWD = S::ROWD, NRS = S::NRS, NSET = S::NSET, ND = S::ND;
    static_assert(NW % WT == 0 && (!FOLD || (ND % 2 == 0)), "even-degree and odd-degree warps come in pairs");
    static_assert(TL == SHT_TQ, "the block's degrees must be one kappa quantum");
    extern __shared__ __align__(128) unsigned char smem_raw[];
    S& sm = *reinterpret_cast<S*>(smem_raw);

    // blocks are dispatched in linear order: tile-major, pass-minor, so that the heavy (large-l) tiles of EVERY pass start first
    const unsigned bid = blockIdx.x + gridDim.x * blockIdx.y, tile = bid / gridDim.y;
    const ThetaPass P = A.passes[bid % gridDim.y];
    const int ntt = A.ntp / NTH, nlt = A.Lp / TL;
    const int lt = nlt - 1 - (int)(tile / ntt), tt = tile % ntt;
    const int l0 = lt * TL, th0 = tt * NTH;
    const int an = P.n < 0 ? -P.n : P.n;
    if (l0 + TL <= an || l0 >= A.L || th0 >= A.nth || th0 + NTH <= A.th_lo || th0 >= A.th_hi) return;
    const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
    int mtop = min(l0 + TL - 1, A.L - 1);
    const int m_end = P.m_end;
    int npairs = (mtop - m_end + 2) / KS;             // an odd step count ends with a dummy step m_end-1 (all-zero table row)
    int pbeg, pend;
    if (!skip_range<SM>(A, bid, npairs, pbeg, pend)) return;
    // the loops below count pairs from 0 at step mtop, as if the tile started where its silent head ends (pbeg is a multiple of 8, so the
    // ring slots and mbarrier phases derived from the pair counter are the same)
    mtop -= KS * pbeg; npairs = pend - pbeg;

    if (tid == 0) {
        for (int i = 0; i < NST; ++i) mbar_init(&sm.full[i], 1);
        for (int i = 0; i < NRS; ++i) { mbar_init(&sm.rfull[i], NW); mbar_init(&sm.rempty[i], NAUX); }
        mbar_fence_init();
    }
    __syncthreads();

    if (w >= NW) {
        // ---------------------------------------------------------------- auxiliary warps: TMA producer + reducers
        reg_dealloc_aux<(FOLD && NC == 2) ? 56 : 40>();
        const int at = tid - NW * 32;                 // 0..127: owns output pairs (re, im) at, at+128, ... of the NOUT per step
        constexpr int NOUT = NTH * NC, NQ = (NOUT + NAUX * 32 - 1) / (NAUX * 32);
        constexpr uint32_t op_bytes = TL * ROWD * sizeof(double), lam_bytes = NTH * sizeof(double);
        auto issue = [&](int p) {
            const int m = mtop - KS * p, slot = p & (NST - 1);
            mbar_expect_tx(&sm.full[slot], KS * (op_bytes + lam_bytes));
#pragma unroll
            for (int h = 0; h < KS; ++h) {
                const size_t row = (size_t)(m - h - m_end + 1);      // table rows start at m_end-1
                bulk_g2s(&sm.op[slot][h][0], P.in + (row * A.Lp + l0) * ROWD, op_bytes, &sm.full[slot]);
                bulk_g2s(&sm.lam[slot][h][0], P.lam + row * A.ntp + th0, lam_bytes, &sm.full[slot]);
            }
        };
        if (at == 0)
            for (int p = 0; p < NST && p < npairs; ++p) issue(p);
        int mlo[NQ], wtq[NQ];                         // wtq: ring group of the output's ring (which warp of a degree group wrote it)
        bool valid[NQ], neg[NQ], south[NQ];
        double* obase[NQ];
        ptrdiff_t osouth[NQ];                         // FOLD: offset (doubles) from the ring's entry to its mirror ring's
#pragma unroll
        for (int q = 0; q < NQ; ++q) {
            const int o = at + NAUX * 32 * q;
            const int th = th0 + o % NTH;             // partial sums are stored [column][ring]
            wtq[q] = (o % NTH) / (32 * RT);
            neg[q] = NC == 2 && (o / NTH);
            valid[q] = th < A.nth && o < NOUT && th >= A.th_lo && th < A.th_hi;
            mlo[q] = P.m_lo ? P.m_lo[th] : -(1 << 30);
            if (mlo[q] < m_end) mlo[q] = m_end;
            // fold pass (n != 0, ring set symmetric about the equator): the -m column is F_{-m} of the MIRRORED ring pi - theta, served by the
            // same d-value (d^l_{-m,n}(pi - theta) = (-1)^{l-n} d^l_{m,n}(theta); the sign rides on the operand) for m > m_s(theta)
            if (NC == 2 && P.fold && neg[q]) mlo[q] += 1;
            obase[q] = reinterpret_cast<double*>(P.out) + (size_t)((NC == 2 && P.fold && neg[q] && th < A.nth) ? A.nth - 1 - th : th) * 2;
            const int tm = A.nfull - 1 - th;
            south[q] = FOLD && tm != th;              // the equator ring of an odd ring count mirrors itself
            osouth[q] = ((ptrdiff_t)tm - th) * 2;
        }
        for (int p = 0; p < npairs; ++p) {
            const int rs = p & (NRS - 1);
            mbar_wait(&sm.rfull[rs], (p / NRS) & 1);
            if (SM == 1 && at == 0) {                  // probe: first pair, 8 steps below the ramp or later, in which any warp contributed
                int fl = 0;
#pragma unroll
                for (int ww = 0; ww < NW; ++ww) fl |= sm.act[rs][ww] & 4;
                if (p == 0) A.skip_p0[bid] = 1 << 30;
                if (fl && mtop - KS * p < l0 - 8 && A.skip_p0[bid] == (1 << 30)) A.skip_p0[bid] = p;
            }
            int actb[ND][NQ];                          // flags of the warp that wrote output q of degree group ww
#pragma unroll
            for (int ww = 0; ww < ND; ++ww)
#pragma unroll
                for (int q = 0; q < NQ; ++q) actb[ww][q] = sm.act[rs][ww * WT + wtq[q]];
#pragma unroll
            for (int h = 0; h < KS; ++h) {
                const int m = mtop - KS * p - h;
                double2 v[NSET][NQ];
#pragma unroll
                for (int e = 0; e < NSET; ++e)
#pragma unroll
                    for (int q = 0; q < NQ; ++q) v[e][q] = make_double2(0.0, 0.0);
                bool any = false;
#pragma unroll
                for (int ww = 0; ww < ND; ++ww) {
                    const int es = FOLD ? (ww & 1) : 0;           // FOLD: degree group ww carries degrees of parity ww & 1
                    const double2* r = reinterpret_cast<const double2*>(&sm.red[rs][h][ww][0][0]) + at;
#pragma unroll
                    for (int q = 0; q < NQ; ++q)
                        if (at + NAUX * 32 * q < NOUT && ((actb[ww][q] >> h) & 1)) {
                            any = true;
                            const double2 t = r[NAUX * 32 * q];
                            if (FOLD && es) { v[NSET - 1][q].x += t.x; v[NSET - 1][q].y += t.y; }
                            else { v[0][q].x += t.x; v[0][q].y += t.y; }
                        }
                }
                if (any) {
#pragma unroll
                    for (int q = 0; q < NQ; ++q) {
                        if (valid[q] && m >= mlo[q] && !(neg[q] && m == 0 && !P.fold)) {
                            const int m_out = (NC == 2) ? (neg[q] ? -m : m) : P.sgn_out * m;
                            const int row = m_out < 0 ? m_out + A.NB : m_out;
                            double* o = obase[q] + (size_t)row * A.ldout * 2;
                            if (FOLD) {
                                // set 0 = degrees of even l (la is even): E if m is even, O if m is odd
                                const double2 a = v[0][q], b = v[NSET - 1][q];
                                red_add_f64(o, a.x + b.x); red_add_f64(o + 1, a.y + b.y);                    // F_m(theta) = E + O
                                if (south[q]) {
                                    const double sg = (m & 1) ? -1.0 : 1.0;                                     // F_m(pi - theta) = E - O
                                    red_add_f64(o + osouth[q], sg * (a.x - b.x)); red_add_f64(o + osouth[q] + 1, sg * (a.y - b.y));
                                }
                            } else {
                                red_add_f64(o, v[0][q].x); red_add_f64(o + 1, v[0][q].y);
                            }
                        }
                    }
                }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(&sm.rempty[rs]);
            if (at == 0 && p + NST < npairs) issue(p + NST);   // every compute warp has finished pair p: its slot is free
        }
        return;
    }
    reg_alloc_compute<(FOLD && NC == 2) ? 56 : 40>();

    // -------------------------------------------------------------------- compute warps
    // degrees of this warp: la + DS j, j < RL (FOLD: one parity per warp, DS = 2)
    constexpr int DS = FOLD ? 2 : 1;
    const int wd = w / WT, tho = (w % WT) * 32 * RT;  // degree group; first ring of the warp inside the block's ring tile
    const int la = FOLD ? l0 + 2 * RL * (wd >> 1) + (wd & 1) : l0 + wd * RL, l_hi = la + DS * (RL - 1);
    const bool warp_real = la < A.L;
    double cur[NI], prev[NI];
    KPack<NI> kp;
    kp.fill(0xffffffffu);
#pragma unroll
    for (int q = 0; q < NI; ++q) { cur[q] = 0.0; prev[q] = 0.0; }
    bool wact = false;                                // some item of this warp has k == 0 (its contribution matters)
    const double* stv = P.st_val + (size_t)la * A.ntp + th0 + tho + lane;
    const uint8_t* stk = P.st_k + (size_t)la * A.ntp + th0 + tho + lane;

    // one recursion step; `ca` holds e_m, `cb` holds e_{m+1} on entry and e_{m-1} on exit (roles swap every step, so the
    // iterates never move between registers).  Returns true if partial sums were written.
    auto step = [&](const int m, const int slot, const int rs, const int h, double (&ca)[NI],
                    double (&cb)[NI]) -> bool {
        if (!(m <= l_hi && warp_real)) return false;
        bool wrote = false;
        if (m >= la) {                                // the degree l == m starts (warp-uniform): Eq. 27 start values
            if (DS == 1 || ((m - la) & 1) == 0) {     // (one address computed here, not RL row pointers kept in registers)
                const size_t so = (size_t)(m - la) * A.ntp;
                double sv[RT]; uint32_t sk[RT];
#pragma unroll
                for (int i = 0; i < RT; ++i) { sv[i] = stv[so + 32 * i]; sk[i] = stk[so + 32 * i]; }
#pragma unroll
                for (int j = 0; j < RL; ++j) {
                    if (m == la + DS * j) {
#pragma unroll
                        for (int i = 0; i < RT; ++i) {
                            ca[j * RT + i] = sv[i];
                            cb[j * RT + i] = 0.0;
                            kp.set(j * RT + i, sk[i]);
                        }
                    }
                }
            }
            wact = true;                              // re-evaluated at the next window check
        }
        const double* row = &sm.op[slot][h][(la - l0) * ROWD];
        const double s = row[ROWD - 1];
        double lam[RT];
#pragma unroll
        for (int i = 0; i < RT; ++i) lam[i] = sm.lam[slot][h][tho + lane + 32 * i] * s;
        if (wact) {
            double acc[RT][2 * NC];
#pragma unroll
            for (int i = 0; i < RT; ++i)
#pragma unroll
                for (int c = 0; c < 2 * NC; ++c) acc[i][c] = 0.0;
#pragma unroll
            for (int j = 0; j < RL; ++j) {
                const double* r = row + (DS * j) * ROWD;
                double cf[2 * NC];
#pragma unroll
                for (int c = 0; c < NC; ++c) {
                    const double2 t = *reinterpret_cast<const double2*>(r + 2 * c);
                    cf[2 * c] = t.x; cf[2 * c + 1] = t.y;
                }
                const double g = r[2 * NC];
#pragma unroll
                for (int i = 0; i < RT; ++i) {
                    const double e = ca[j * RT + i];
#pragma unroll
                    for (int c = 0; c < 2 * NC; ++c) acc[i][c] = fma(e, cf[c], acc[i][c]);
                    cb[j * RT + i] = fma(lam[i], e, -(g * cb[j * RT + i]));
                }
            }
            double2* rd = reinterpret_cast<double2*>(&sm.red[rs][h][wd][0][0]) + tho;
#pragma unroll
            for (int i = 0; i < RT; ++i)
#pragma unroll
                for (int c = 0; c < NC; ++c) rd[c * NTH + lane + 32 * i] = make_double2(acc[i][2 * c], acc[i][2 * c + 1]);
            wrote = true;
        } else {                                      // every item of the warp is still below 2^-340: recursion only
#pragma unroll
            for (int j = 0; j < RL; ++j) {
                const double g = row[(DS * j) * ROWD + 2 * NC];
#pragma unroll
                for (int i = 0; i < RT; ++i) cb[j * RT + i] = fma(lam[i], ca[j * RT + i], -(g * cb[j * RT + i]));
            }
        }
        if ((m & (SHT_JCHK - 1)) == 0) {
            if (kp.any_nonzero()) window_check<NI>(cb, ca, kp);
            if (P.m_lo) dead_check<NI>(cb, ca);
            if (m < la) wact = __any_sync(0xffffffffu, kp.any_zero_byte());
        }
        return wrote;
    };
    if (SM == 0 && pbeg > 0) skip_load<NI>(A, bid, tid, cur, prev, kp, wact);      // transform: the state the silent head would have produced
    for (int p = 0; p < npairs; ++p) {
        const int m = mtop - KS * p, slot = p & (NST - 1), rs = p & (NRS - 1);
        const uint32_t rparity = ((p / NRS) & 1) ^ 1;
        mbar_wait(&sm.full[slot], (p / NST) & 1);
        // the reducers are done with this hand-off slot (waiting here, not in front of the first partial-sum store, keeps
        // the compute section free of barriers so that operand loads of both steps can be hoisted above the FMAs)
        mbar_wait(&sm.rempty[rs], rparity);
        int flags = 0;
        if (step(m, slot, rs, 0, cur, prev)) flags |= 1;
        if (step(m - 1, slot, rs, 1, prev, cur)) flags |= 2;
        if (SM == 1 && warp_matters<NI>(cur, kp)) flags |= 4;
        __syncwarp();
        if (lane == 0) {
            sm.act[rs][w] = flags;
            mbar_arrive(&sm.rfull[rs]);
        }
    }
    if (SM == 2) skip_store<NI>(A, bid, tid, cur, prev, kp, wact);
}

// =============================================================================================================
// forward theta step, Eq. 30:  H[m_out+L-1][l] += c_m(l) * sum_theta W[m][theta] * e^l_m(theta)
// block tile: TLB = 32*RL degrees x NTB = NW*RT rings; KS = 2 recursion steps per pipeline stage
// =============================================================================================================
// FOLD (n = 0 on a ring set symmetric about the equator): only the northern rings are recursed; d^l_{m,0}(pi - theta) =
// (-1)^{l+m} d^l_{m,0}(theta), so a degree with l+m even contracts with E = W(theta) + W(pi-theta) and one with
// l+m odd with O = W(theta) - W(pi-theta).  Operand rows then hold both sets: [ring][E, O][NC].  A thread's two degrees
// l0 + lane + {0, 32} have the SAME parity, which alternates with the lane: one shared-memory load with two distinct addresses
// (even lanes one set, odd lanes the other) serves both degrees of every lane in a single wavefront -- half the operand
// wavefronts of a mapping whose two degrees differ in parity (the r1 kernel was bound by the shared-memory pipe at 86 %).
template <int RL, int RT, int NW, int NC, bool FOLD>
struct FwdSmem {
    static constexpr int TLB = 32 * RL, NTB = NW * RT, NCW = FOLD ? 2 * NC : NC;
    double2 wt[NST][KS][NTB * NCW];         // weighted F_m samples of the block's rings (TMA ring)
    double lamraw[NST][KS][NTB];            // lambda_m(theta) (TMA ring)
    double2 sg[NST][KS];                    // (s, G) of the block's quantum: [KS-1-h] belongs to step h of the pair
    double hdr[NW][KS][RT];                 // lambda'_m = lambda_m s_m of each warp's own rings
    double red[NRS][KS][NW][TLB][2 * NC];   // per-warp partial sums
    int act[NRS][NW];
    uint64_t full[NST], rfull[NRS], rempty[NRS];
};

template <int RL, int RT, int NW, int NC, bool FOLD, int SM>
__global__ void __launch_bounds__((NW + NAUX) * 32, 1) theta_forward_kernel(const ThetaArgs A) {
    using S = FwdSmem<RL, RT, NW, NC, FOLD>;
    constexpr int TLB = S::TLB, NTB = S::NTB, NI = RL * RT, NCW = S::NCW;
    static_assert(RL == 2, "two degrees of opposite parity per thread");
    static_assert(TLB == SHT_TQ, "the block's degrees must be one kappa quantum");
    static_assert(KS * RT <= 32, "one lane per lambda' value of a pair");
    extern __shared__ __align__(128) unsigned char smem_raw[];
    S& sm = *reinterpret_cast<S*>(smem_raw);

    const unsigned bid = blockIdx.x + gridDim.x * blockIdx.y, tile = bid / gridDim.y;      // tile-major, pass-minor (see the inverse kernel)
    const ThetaPass P = A.passes[bid % gridDim.y];
    const int ntt = A.ntp / NTB, nlt = A.Lp / TLB;
    const int lt = nlt - 1 - (int)(tile / ntt), tt = tile % ntt;
    const int l0 = lt * TLB, th0 = tt * NTB;
    const int an = P.n < 0 ? -P.n : P.n;
    if (l0 + TLB <= an || l0 >= A.L || th0 >= A.nth || th0 + NTB <= A.th_lo || th0 >= A.th_hi) return;   // (rings outside the shard inside a
                                                                                                       //  boundary tile carry zero operands)
    const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
    int mtop = min(l0 + TLB - 1, A.L - 1);
    const int m_end = P.m_end;
    int npairs = (mtop - m_end + 2) / KS;
    int pbeg, pend;
    if (!skip_range<SM>(A, bid, npairs, pbeg, pend)) return;
    mtop -= KS * pbeg; npairs = pend - pbeg;           // pairs count from 0 at the step the silent head ends (see the inverse kernel)

    if (tid == 0) {
        for (int i = 0; i < NST; ++i) mbar_init(&sm.full[i], 1);
        for (int i = 0; i < NRS; ++i) { mbar_init(&sm.rfull[i], NW); mbar_init(&sm.rempty[i], NAUX); }
        mbar_fence_init();
    }
    __syncthreads();

    if (w >= NW) {
        // ---------------------------------------------------------------- auxiliary warps
        reg_dealloc_aux<(NC == 1 && RT == 16) ? 56 : 40>();
        const int at = tid - NW * 32;
        constexpr int NOUT = TLB * NC, NQ = (NOUT + NAUX * 32 - 1) / (NAUX * 32);
        constexpr uint32_t wt_bytes = NTB * NCW * sizeof(double2), lam_bytes = NTB * sizeof(double);
        const double2* sgrow = A.sg + (size_t)lt * A.sgstride - A.mmin;
        auto issue = [&](int p) {
            const int m = mtop - KS * p, slot = p & (NST - 1);
            mbar_expect_tx(&sm.full[slot], KS * (wt_bytes + lam_bytes + (uint32_t)sizeof(double2)));
#pragma unroll
            for (int h = 0; h < KS; ++h) {
                const size_t row = (size_t)(m - h - m_end + 1);
                bulk_g2s(&sm.wt[slot][h][0], P.in + (row * A.ntp + th0) * 2 * NCW, wt_bytes, &sm.full[slot]);
                bulk_g2s(&sm.lamraw[slot][h][0], P.lam + row * A.ntp + th0, lam_bytes, &sm.full[slot]);
            }
            bulk_g2s(&sm.sg[slot][0], sgrow + (m - KS + 1), KS * (uint32_t)sizeof(double2), &sm.full[slot]);
        };
        if (at == 0)
            for (int p = 0; p < NST && p < npairs; ++p) issue(p);
        int lq[NQ];
        bool valid[NQ], neg[NQ];
        double* obase[NQ];
        double osgn[NQ];                              // fold passes: (-1)^{l-n} on the -m column (internal.h)
#pragma unroll
        for (int q = 0; q < NQ; ++q) {
            const int o = at + NAUX * 32 * q;
            lq[q] = l0 + o % TLB;                     // partial sums are stored [column][degree]
            neg[q] = NC == 2 && (o / TLB);
            valid[q] = o < NOUT && lq[q] >= an && lq[q] < A.L;
            if (o >= NOUT) lq[q] = l0;
            obase[q] = reinterpret_cast<double*>(P.out) + (size_t)lq[q] * 2;
            osgn[q] = (P.fold && neg[q] && ((lq[q] - P.n) & 1)) ? -1.0 : 1.0;
        }
        // c_m(l) of the owned degrees, fetched one pair ahead (coalesced rows of the plan-time table)
        const double* crow = A.ctab + (size_t)(mtop - A.mmin) * A.Lp;
        double cn[KS][NQ];
#pragma unroll
        for (int h = 0; h < KS; ++h)
#pragma unroll
            for (int q = 0; q < NQ; ++q) cn[h][q] = crow[-(ptrdiff_t)h * A.Lp + lq[q]];
        for (int p = 0; p < npairs; ++p) {
            const int rs = p & (NRS - 1);
            double cm[KS][NQ];
#pragma unroll
            for (int h = 0; h < KS; ++h)
#pragma unroll
                for (int q = 0; q < NQ; ++q) cm[h][q] = cn[h][q];
            if (p + 1 < npairs) {
                crow -= (size_t)KS * A.Lp;
#pragma unroll
                for (int h = 0; h < KS; ++h)
#pragma unroll
                    for (int q = 0; q < NQ; ++q) cn[h][q] = crow[-(ptrdiff_t)h * A.Lp + lq[q]];
            }
            mbar_wait_relaxed(&sm.rfull[rs], (p / NRS) & 1);      // (forward: -0.7 ... -1.5 % with the back-off; the inverse reducers are on the critical path: +2 %)
            int actb[NW];
#pragma unroll
            for (int ww = 0; ww < NW; ++ww) actb[ww] = sm.act[rs][ww];
            if (SM == 1 && at == 0) {                  // probe (see the inverse kernel)
                int fl = 0;
#pragma unroll
                for (int ww = 0; ww < NW; ++ww) fl |= actb[ww] & 4;
                if (p == 0) A.skip_p0[bid] = 1 << 30;
                if (fl && mtop - KS * p < l0 - 8 && A.skip_p0[bid] == (1 << 30)) A.skip_p0[bid] = p;
            }
#pragma unroll
            for (int h = 0; h < KS; ++h) {
                const int m = mtop - KS * p - h;
                double2 v[NQ];
#pragma unroll
                for (int q = 0; q < NQ; ++q) v[q] = make_double2(0.0, 0.0);
                bool any = false;
#pragma unroll
                for (int ww = 0; ww < NW; ++ww) {
                    if ((actb[ww] >> h) & 1) {
                        any = true;
                        const double2* r = reinterpret_cast<const double2*>(&sm.red[rs][h][ww][0][0]);
#pragma unroll
                        for (int q = 0; q < NQ; ++q) {
                            const int o = at + NAUX * 32 * q;
                            if (o < NOUT) { const double2 t = r[o]; v[q].x += t.x; v[q].y += t.y; }
                        }
                    }
                }
                if (any && m >= m_end) {
#pragma unroll
                    for (int q = 0; q < NQ; ++q) {
                        // (the -m column of a plain PM pass is all zero at m = 0: its operand is zeroed by the weight split)
                        if (valid[q] && lq[q] >= m && lq[q] >= -m) {
                            const int m_out = (NC == 2) ? (neg[q] ? -m : m) : P.sgn_out * m;
                            double* o = obase[q] + (size_t)(m_out + A.L - 1) * A.Lp * 2;
                            const double cmq = cm[h][q] * osgn[q];
                            red_add_f64(o, v[q].x * cmq); red_add_f64(o + 1, v[q].y * cmq);
                        }
                    }
                }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(&sm.rempty[rs]);
            if (at == 0 && p + NST < npairs) issue(p + NST);
        }
        return;
    }
    reg_alloc_compute<(NC == 1 && RT == 16) ? 56 : 40>();

    // -------------------------------------------------------------------- compute warps
    // state: start values preloaded; a lane holds still (lambda' = 1, g' = 0) until m reaches its degree
    double cur[NI], prev[NI], x[RL];
    KPack<NI> kp;
    int lr[RL];
#pragma unroll
    for (int r = 0; r < RL; ++r) {
        lr[r] = l0 + lane + 32 * r;                    // the thread's degrees share their parity (FOLD: one operand set for both)
        const bool ok = lr[r] >= an && lr[r] < A.L;
        x[r] = (double)(lr[r] - mtop) * (double)(lr[r] + mtop + 1);
#pragma unroll
        for (int i = 0; i < RT; ++i) {
            const size_t o = (size_t)lr[r] * A.ntp + th0 + w * RT + i;
            cur[r * RT + i] = ok ? P.st_val[o] : 0.0;
            prev[r * RT + i] = 0.0;
            kp.set(r * RT + i, ok ? (uint32_t)P.st_k[o] : 0u);
        }
    }
    double tm = 2.0 * (double)mtop;                    // x_{m-1} = x_m + 2m
    bool wact = true;
    if (SM == 0 && pbeg > 0) {                         // transform: the state the silent head would have produced, at step m0
        skip_load<NI>(A, bid, tid, cur, prev, kp, wact);   // (x and tm above are already those of the step the head ends at)
    }

    // one recursion step; `ca` holds e_m, `cb` holds e_{m+1} on entry and e_{m-1} on exit (roles swap every step)
    auto step = [&](const int m, const int slot, const int rs, const int h, double (&ca)[NI],
                    double (&cb)[NI]) -> bool {
        // operand set of the thread's degrees: FOLD picks E (l+m even) or O (l+m odd) by address, per lane parity
        const double2* Tq = &sm.wt[slot][h][w * RT * NCW] + (FOLD ? ((l0 + m + lane) & 1) * NC : 0);
        const double* LM = &sm.hdr[w][h][0];
        const double G = sm.sg[slot][KS - 1 - h].y;
        bool wrote = false;
        double acc[RL][2 * NC];
#pragma unroll
        for (int r = 0; r < RL; ++r)
#pragma unroll
            for (int c = 0; c < 2 * NC; ++c) acc[r][c] = 0.0;
        if (m >= l0) {
            // ---- ramp: lanes whose degree is still above m hold still
            double g[RL]; bool on[RL];
#pragma unroll
            for (int r = 0; r < RL; ++r) { on[r] = m <= lr[r]; g[r] = on[r] ? x[r] * G : 0.0; }
#pragma unroll
            for (int i = 0; i < RT; ++i) {
                const double lm = LM[i];
                const double2 w0 = Tq[i * NCW];
                double2 w1 = make_double2(0.0, 0.0);
                if (NC == 2) w1 = Tq[i * NCW + 1];
#pragma unroll
                for (int r = 0; r < RL; ++r) {
                    const double e = ca[r * RT + i];
                    acc[r][0] = fma(e, w0.x, acc[r][0]); acc[r][1] = fma(e, w0.y, acc[r][1]);
                    if (NC == 2) { acc[r][2] = fma(e, w1.x, acc[r][2]); acc[r][3] = fma(e, w1.y, acc[r][3]); }
                    cb[r * RT + i] = fma(on[r] ? lm : 1.0, e, -(g[r] * cb[r * RT + i]));     // off: copies the start value
                    ca[r * RT + i] = on[r] ? e : 0.0;                                         //      and keeps e_{m+1} = 0
                }
            }
            wrote = true;
        } else if (wact) {
            double g[RL];
#pragma unroll
            for (int r = 0; r < RL; ++r) g[r] = x[r] * G;
#pragma unroll
            for (int i = 0; i < RT; i += 2) {
                const double2 lm2 = *reinterpret_cast<const double2*>(LM + i);
#pragma unroll
                for (int ii = 0; ii < 2; ++ii) {
                    const double lm = ii ? lm2.y : lm2.x;
                    const double2 w0 = Tq[(i + ii) * NCW];
                    double2 w1 = make_double2(0.0, 0.0);
                    if (NC == 2) w1 = Tq[(i + ii) * NCW + 1];
#pragma unroll
                    for (int r = 0; r < RL; ++r) {
                        const double e = ca[r * RT + i + ii];
                        acc[r][0] = fma(e, w0.x, acc[r][0]); acc[r][1] = fma(e, w0.y, acc[r][1]);
                        if (NC == 2) { acc[r][2] = fma(e, w1.x, acc[r][2]); acc[r][3] = fma(e, w1.y, acc[r][3]); }
                        cb[r * RT + i + ii] = fma(lm, e, -(g[r] * cb[r * RT + i + ii]));
                    }
                }
            }
            wrote = true;
        } else {                                      // every item of the warp is still below 2^-340: recursion only
            double g[RL];
#pragma unroll
            for (int r = 0; r < RL; ++r) g[r] = x[r] * G;
#pragma unroll
            for (int i = 0; i < RT; ++i) {
                const double lm = LM[i];
#pragma unroll
                for (int r = 0; r < RL; ++r) cb[r * RT + i] = fma(lm, ca[r * RT + i], -(g[r] * cb[r * RT + i]));
            }
        }
#pragma unroll
        for (int r = 0; r < RL; ++r) x[r] += tm;
        tm -= 2.0;
        if ((m & (SHT_JCHK - 1)) == 0) {
            if (kp.any_nonzero()) window_check<NI>(cb, ca, kp);
            if (P.m_lo) dead_check<NI>(cb, ca);
            if (m < l0) wact = __any_sync(0xffffffffu, kp.any_zero_byte());
        }
        if (wrote) {
            double2* rd = reinterpret_cast<double2*>(&sm.red[rs][h][w][0][0]);
#pragma unroll
            for (int r = 0; r < RL; ++r)
#pragma unroll
                for (int c = 0; c < NC; ++c) {
                    rd[c * TLB + lane + 32 * r] = make_double2(acc[r][2 * c], acc[r][2 * c + 1]);      // slot = degree - l0; conflict-free
                }
        }
        return wrote;
    };
    for (int p = 0; p < npairs; ++p) {
        const int m = mtop - KS * p, slot = p & (NST - 1), rs = p & (NRS - 1);
        const uint32_t rparity = ((p / NRS) & 1) ^ 1;
        mbar_wait(&sm.full[slot], (p / NST) & 1);
        mbar_wait(&sm.rempty[rs], rparity);
        // lambda' of this warp's rings for both steps of the pair: lane -> (step h, ring i)
        if (lane < KS * RT) {
            const int h = lane / RT, i = lane % RT;
            sm.hdr[w][h][i] = sm.lamraw[slot][h][w * RT + i] * sm.sg[slot][KS - 1 - h].x;
        }
        __syncwarp();
        int flags = 0;
        if (step(m, slot, rs, 0, cur, prev)) flags |= 1;
        if (step(m - 1, slot, rs, 1, prev, cur)) flags |= 2;
        if (SM == 1 && warp_matters<NI>(cur, kp)) flags |= 4;
        __syncwarp();
        if (lane == 0) {
            sm.act[rs][w] = flags;
            mbar_arrive(&sm.rfull[rs]);
        }
    }
    if (SM == 2) skip_store<NI>(A, bid, tid, cur, prev, kp, wact);
}

template <int RL, int RT, int NW, int NC, bool FOLD = false, int WT = 1>
cudaError_t launch_inv(const ThetaArgs& a, cudaStream_t st) {
    using S = InvSmem<RL, RT, NW, NC, FOLD, WT>;
    const size_t smem = sizeof(S) + 128;
    dim3 grid((a.Lp / S::TL) * (a.ntp / S::NTH), a.npass);
    auto k = a.skip_mode == 1 ? theta_inverse_kernel<RL, RT, NW, NC, FOLD, WT, 1>
           : a.skip_mode == 2 ? theta_inverse_kernel<RL, RT, NW, NC, FOLD, WT, 2> : theta_inverse_kernel<RL, RT, NW, NC, FOLD, WT, 0>;
    cudaError_t e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    k<<<grid, (NW + NAUX) * 32, smem, st>>>(a);
    count_launch();
    return cudaGetLastError();
}
template <int RL, int RT, int NW, int NC, bool FOLD>
cudaError_t launch_fwd(const ThetaArgs& a, cudaStream_t st) {
    using S = FwdSmem<RL, RT, NW, NC, FOLD>;
    const size_t smem = sizeof(S) + 128;
    auto k = a.skip_mode == 1 ? theta_forward_kernel<RL, RT, NW, NC, FOLD, 1>
           : a.skip_mode == 2 ? theta_forward_kernel<RL, RT, NW, NC, FOLD, 2> : theta_forward_kernel<RL, RT, NW, NC, FOLD, 0>;
    cudaError_t e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    dim3 grid((a.Lp / S::TLB) * (a.ntp / S::NTB), a.npass);
    k<<<grid, (NW + NAUX) * 32, smem, st>>>(a);
    count_launch();
    return cudaGetLastError();
}

}  // namespace

// Tile shapes: inverse 64 degrees x 128 rings per block: 8 compute warps, 8 degrees x 4 rings per thread (one order per step, P mode) or
//              16 degrees x 2 rings per thread with the warps split 4 degree groups x 2 ring groups (+-m per step, PM mode: measured
//              5-6 % faster there -- L = 8192 inverse 84.7 -> 79.8 ms -- and 1-4 % slower in P mode; 4 ring groups: 15 % slower);
//              forward 64 degrees x 128 rings per block (8 compute warps, 2 degrees x 16 rings per thread).
int theta_inverse_rowd(int mode) { return mode == 0 ? 6 : 4; }
// Tile choice.  A launch has (Lp/64) x (ntp/rings_per_block) x npass blocks whose step counts grow linearly with the degree
// tile, and the longest block alone runs ~L steps.  When 64 x 128 tiles do not even give one block per SM the launch is bound by
// that longest block while the other SMs idle; 64 x 64 tiles then halve the work per step of every block (measured: L = 512
// spin 0 inverse 0.456 -> 0.275 ms, L = 1024 spin 0 inverse 0.906 -> 0.548 ms; with more blocks than SMs the big tile wins).
// ThetaArgs::tile = 64 / 128 (plan option) overrides.
static bool small_tiles(const ThetaArgs& a, int big) {
    if (a.tile) return a.tile == 64;
    const long blocks = (long)(a.Lp / SHT_TQ) * (a.ntp / big) * a.npass;
    return blocks <= a.nsm;
}
// rings per block tile the launchers below choose for these arguments (the plan sizes its per-block skip tables with it)
int theta_tile_rings(const ThetaArgs& a) { return small_tiles(a, 128) ? 64 : 128; }
cudaError_t launch_theta_inverse(const ThetaArgs& a, int mode, cudaStream_t st) {
    if (a.npass == 0) return cudaSuccess;
    if (a.fold0) {
        if (small_tiles(a, 128)) return mode == 0 ? launch_inv<8, 2, 8, 2, true>(a, st) : launch_inv<8, 2, 8, 1, true>(a, st);
        if (mode != 0) return launch_inv<8, 4, 8, 1, true>(a, st);
        return a.tile == 128 ? launch_inv<8, 4, 8, 2, true>(a, st) : launch_inv<16, 2, 8, 2, true, 2>(a, st);
    }
    if (small_tiles(a, 128)) return mode == 0 ? launch_inv<8, 2, 8, 2>(a, st) : launch_inv<8, 2, 8, 1>(a, st);
    if (mode != 0) return launch_inv<8, 4, 8, 1>(a, st);
    return a.tile == 128 ? launch_inv<8, 4, 8, 2>(a, st) : launch_inv<16, 2, 8, 2, false, 2>(a, st);
}
cudaError_t launch_theta_forward(const ThetaArgs& a, int mode, cudaStream_t st) {
    if (a.npass == 0) return cudaSuccess;
    if (small_tiles(a, 128)) {
        if (a.fold0) return mode == 0 ? launch_fwd<2, 8, 8, 2, true>(a, st) : launch_fwd<2, 8, 8, 1, true>(a, st);
        return mode == 0 ? launch_fwd<2, 8, 8, 2, false>(a, st) : launch_fwd<2, 8, 8, 1, false>(a, st);
    }
    if (a.fold0) return mode == 0 ? launch_fwd<2, 16, 8, 2, true>(a, st) : launch_fwd<2, 16, 8, 1, true>(a, st);
    return mode == 0 ? launch_fwd<2, 16, 8, 2, false>(a, st) : launch_fwd<2, 16, 8, 1, false>(a, st);
}
