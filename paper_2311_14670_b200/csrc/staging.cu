// staging.cu -- everything around the hot kernels that is O(L^2): plan-time tables (ring constants, Eq. 27 start
// values in windowed mantissa/exponent form, kappa exponents, quadrature weights) and the per-transform staging
// kernels (layout changes, l-scaling, MW torus extension / upsampling phases, pole ring
// (Eq. 28-29), Hermitian fills).  All of it is HBM-bound and timed separately from the hot path.
#include "staging.h"

#include <math.h>

namespace {

__device__ __forceinline__ double sgn_pow(int k) { return (k & 1) ? -1.0 : 1.0; }

// F_m on quadrature ring ts, read from the forward ring-sample array U.
//   pair = 0: U[bin(m)][ldin], one row per order.
//   pair != 0 (MW / MWSS upsampling, api.cu mw_upsample): the extension of F_m to the theta circle has the reflection symmetry
//   F_m(2pi - theta) = (-1)^{m-n} F_m(theta), which alternates with m.  Row j of U then holds the SUM of the theta-circle
//   samples (ldin = 4L midpoints theta'_u; the mirror of u is ldin-1-u) of the orders m = 2j-(L-1) and 2j-(L-2) -- one even and one odd
//   function, carried through the (linear) FFT upsampling as ONE column -- and either is recovered from its own symmetry:
//   F_m(theta'_u) = (c[u] + (-1)^{m-n} c[ldin-1-u]) / 2.  Half the theta FFT work of the forward transform.
__device__ __forceinline__ double2 u_get(const double2* __restrict__ U, int ldin, int NBin, int pair, int L, int n, int m, int ts) {
    if (!pair) return U[(size_t)(m < 0 ? m + NBin : m) * ldin + ts];
    const double2* row = U + (size_t)((m + L - 1) >> 1) * ldin;
    const double2 a = row[ts], b = row[ldin - 1 - ts];
    const double s = ((m - n) & 1) ? -0.5 : 0.5;
    return make_double2(fma(s, b.x, 0.5 * a.x), fma(s, b.y, 0.5 * a.y));
}

// ---- double-double helpers for the start-value product -------------------------------------------------------
struct dd { double hi, lo; };
__device__ __forceinline__ dd dd_mul(dd a, dd b) {
    double p = a.hi * b.hi;
    double e = fma(a.hi, b.hi, -p);
    e = fma(a.hi, b.lo, e);
    e = fma(a.lo, b.hi, e);
    double s = p + e;
    return {s, e - (s - p)};
}

// Eq. 27 for all l at one ring, as the running product
//   d^l_{l,n} = d^{l-1}_{l-1,n} * ( -sqrt(2l(2l-1)/((l+n)(l-n))) * sin(b/2)cos(b/2) ),   d^{|n|}_{|n|,n} = c2^{2n} or s2^{-2n},
// carried as double-double mantissa * 2^e so that neither the 1e-35000 magnitudes nor l-fold rounding matter
// (R7).  Output: windowed value val = d * 2^(SWIN*k), k = floor((TWIN - e)/SWIN) if e < TWIN else 0.
__global__ void k_start_values(int L, int n, int nth, int ntp, const double* __restrict__ c2hi, const double* __restrict__ c2lo,
                               const double* __restrict__ s2hi, const double* __restrict__ s2lo, const double* __restrict__ rhi,
                               const double* __restrict__ rlo, double* __restrict__ st_val, uint8_t* __restrict__ st_k,
                               int* __restrict__ range_flag) {
    int th = blockIdx.x * blockDim.x + threadIdx.x;
    if (th >= nth) return;
    const int an = n < 0 ? -n : n;
    dd c = {c2hi[th], c2lo[th]}, s = {s2hi[th], s2lo[th]};
    dd q = dd_mul(c, s);
    q.hi = -q.hi; q.lo = -q.lo;
    dd base = n >= 0 ? c : s;
    dd v = {1.0, 0.0};
    long e = 0;
    for (int i = 0; i < 2 * an; ++i) {
        v = dd_mul(v, base);
        int ex; double f = frexp(v.hi, &ex);
        v.hi = f; v.lo = ldexp(v.lo, -ex); e += ex;
    }
    for (int l = an; l < L; ++l) {
        if (l > an) {
            dd r = {rhi[l], rlo[l]};
            v = dd_mul(dd_mul(v, r), q);
            int ex; double f = frexp(v.hi, &ex);
            v.hi = f; v.lo = ldexp(v.lo, -ex); e += ex;
        }
        long k = 0;
        if (e < SHT_TWIN) k = (SHT_TWIN - e) / SHT_SWIN;
        if (k > 254) {      // below 2^-122900: outside the one-byte window counter.  The iterate would grow back to O(1) at small m,
            *range_flag = 1;   // so the value must not be dropped: the plan is refused (api.cu check_start_range / set_workspace)
            st_val[(size_t)l * ntp + th] = 0.0; st_k[(size_t)l * ntp + th] = 0; continue;
        }
        st_val[(size_t)l * ntp + th] = ldexp(v.hi + v.lo, (int)(e + k * SHT_SWIN));
        st_k[(size_t)l * ntp + th] = (uint8_t)k;
    }
}

// kappa exponents: for a tile with l_top = TQ*(row+1): k_m chosen greedily so that c_m(l_top) = prod a_{j-1}(l_top) 2^{k_j}
// stays in [1,2).  Entry for m = l_top is 0.
__global__ void k_kexp(int nrows, int kstride, int kmin, int8_t* __restrict__ kexp) {
    int row = blockIdx.x * blockDim.x + threadIdx.x;
    if (row >= nrows) return;
    const int ltop = SHT_TQ * (row + 1);
    int8_t* kr = kexp + (size_t)row * kstride - kmin;
    for (int m = kmin; m <= kmin + kstride - 1; ++m) kr[m] = 0;
    double P = 1.0;
    for (int m = ltop; m > kmin && m > -ltop; --m) {
        double x = (double)(ltop - m + 1) * (double)(ltop + m);
        if (x <= 0.0) break;
        P *= 2.0 / sqrt(x);
        int ex; (void)frexp(P, &ex);
        int kk = -(ex - 1);
        if (m <= ltop - 1 || true) kr[m] = (int8_t)kk;
        P = ldexp(P, kk);
    }
}

__global__ void k_rsq(int n, double* __restrict__ rsq) {
    int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k < n) rsq[k] = k > 0 ? 1.0 / sqrt((double)k) : 0.0;
}

// c_m(l) table (internal.h): C[m - mmin][Lp]; c_l = 1, c_{m-1} = c_m a_{m-1}(l) 2^{k_m} = c_m 2^{k_m+1} / sqrt((l-m+1)(l+m)).
// One thread per degree, sequential in m (an O(L^2) plan-time table, independent of the rings and of n).
__global__ void k_ctab(int L, int Lp, int mmin, int kstride, int kmin, const int8_t* __restrict__ kexp,
                       const double* __restrict__ rsq, double* __restrict__ C) {
    int l = blockIdx.x * blockDim.x + threadIdx.x;
    if (l >= Lp) return;
    for (int m = L - 1; m > l || (l >= L && m >= mmin); --m) C[(size_t)(m - mmin) * Lp + l] = 0.0;
    if (l >= L) return;
    const int8_t* kr = kexp + (size_t)(l / SHT_TQ) * kstride - kmin;
    double c = 1.0;
    for (int m = l; m >= mmin; --m) {
        C[(size_t)(m - mmin) * Lp + l] = c;
        if (m > mmin) c = (l + m > 0) ? c * ldexp(1.0, kr[m] + 1) * rsq[l - m + 1] * rsq[l + m] : 0.0;
    }
}
// (s_m, G_m) = (2^{-k_m}, 2^{-2-k_m-k_{m+1}}) per quantum row, column m - mmin
__global__ void k_sgtab(int nrows, int ncol, int mmin, int kstride, int kmin, const int8_t* __restrict__ kexp, double2* __restrict__ SG) {
    int c = blockIdx.x * blockDim.x + threadIdx.x, row = blockIdx.y;
    if (c >= ncol || row >= nrows) return;
    const int m = mmin + c;
    const int8_t* kr = kexp + (size_t)row * kstride - kmin;
    SG[(size_t)row * ncol + c] = make_double2(ldexp(1.0, -kr[m]), ldexp(1.0, -2 - kr[m] - kr[m + 1]));
}
// lambda_m(theta) = (n - m cos theta)/sin theta, evaluated without cancellation (R8) as
// (n - sigma m) csc + m tau;  table [m - m_end][ntp] for one second index n
__global__ void k_lamtab(int n, int nth, int ntp, int m_end, const double* __restrict__ csc, const double* __restrict__ tau,
                         const double* __restrict__ sig, double* __restrict__ lam) {
    int th = blockIdx.x * blockDim.x + threadIdx.x;
    const int m = m_end + blockIdx.y;
    if (th >= ntp) return;
    double v = 0.0;
    if (th < nth) v = fma((double)n - sig[th] * (double)m, csc[th], (double)m * tau[th]);
    lam[(size_t)(m - m_end) * ntp + th] = v;
}

// Theta-quadrature weights of the MW forward transform on the midpoint rings theta'_u = (2u+1)pi/N, N = 4L, u < 2L.
// The integrand G(theta) = F_m(theta) d^l_{m,-s}(theta) is a trigonometric polynomial of degree <= 2L-2, even about 0, so
//   int_0^pi G sin = (1/2) int_0^2pi G |sin| = pi sum_k G^_k c_k,  |sin| = sum_k c_k e^{ik theta}, c_k = (2/pi)/(1-k^2) (k even),
// which is Eq. 41-44 with the reflection sign +1 (R9); G^_k from N samples is exact (N > 4L-4).
// Folding theta <-> 2pi - theta:  v_u = (1/N) (4 + 8 sum_{j=1}^{L-1} cos(2j theta'_u)/(1-4j^2)).   Output: v_u * qphi.
__global__ void k_mid_weights(int L, int count, double qphi, double* __restrict__ w) {
    int u = blockIdx.x * blockDim.x + threadIdx.x;
    if (u >= count) return;
    const long N = 4L * L;
    double acc = 0.0;
    for (int j = L - 1; j >= 1; --j) {              // small terms first
        long r = ((long)2 * j * (2 * u + 1)) % (2 * N);
        acc += 1.0 / (1.0 - 4.0 * (double)j * (double)j) * cospi((double)r / (double)N);
    }
    w[u] = (4.0 + 8.0 * acc) / (double)N * qphi;
}

// MW theta-quadrature weights at band-limit Lq (closed form of Eq. 41-44 with reflection sign +1, R9):
//   v_u = (zeta_u/(2Lq-1)) sum_{|2j|<=Lq-1} 4 cos(2j theta_u)/(1-4j^2),  theta_u = (2u+1)pi/(2Lq-1);  times qphi.
__global__ void k_mw_weights(int Lq, double qphi, double* __restrict__ w) {
    int u = blockIdx.x * blockDim.x + threadIdx.x;
    if (u >= Lq) return;
    const int T = 2 * Lq - 1, jmax = (Lq - 1) / 2;
    double acc = 2.0;                               // j = 0 term: 2/(1-0) * 2 * ... /2 handled below
    acc = 0.0;
    for (int j = jmax; j >= 1; --j) {               // small terms first
        long r = ((long)2 * j * (2 * u + 1)) % (2L * T);
        acc += 4.0 / (1.0 - 4.0 * (double)j * (double)j) * cospi((double)r / (double)T);
    }
    acc = 2.0 * acc + 4.0;                          // +-j pairs, plus j = 0
    double v = acc / (double)T;
    if (u == Lq - 1) v *= 0.5;
    w[u] = v * qphi;
}

// ---- per-transform staging ------------------------------------------------------------------------------------
// inverse prep: coef[l][NB] -> operand rows G[m-m_end][Lp][ROWD] of one pass: {c Re, c Im (x NC), g'_m(l), s_m} with
// c = scale(l) * sign * c_m(l) (internal.h), through a 32x32 shared-memory transpose (coef is l-major, G is m-major).
__global__ void k_prep_inverse(int L, int Lp, int NC, int mmin, const double2* __restrict__ coef_base, size_t coef_slab,
                               const int* __restrict__ cslab, const double* __restrict__ scale, const double* __restrict__ C,
                               const double2* __restrict__ SG, int sgstride, const ThetaPass* __restrict__ passes) {
    // one launch serves all passes of a kernel mode: grid.z = pass (its operand rows start one row into ThetaPass::in)
    const ThetaPass P = passes[blockIdx.z];
    const int n = P.n, sgn_out = P.sgn_out, m_end = P.m_end, fold = P.fold;
    const double2* coef = coef_base + (size_t)cslab[P.slab] * coef_slab;
    double* G = const_cast<double*>(P.in) + (size_t)Lp * (2 * NC + 2);
    if (m_end + (int)blockIdx.y * 32 >= L) return;
    __shared__ double2 tile[2][32][33];
    const int NB = 2 * L - 1, an = n < 0 ? -n : n, ROWD = 2 * NC + 2;
    const int l0 = blockIdx.x * 32, m0 = m_end + blockIdx.y * 32;
    for (int c = 0; c < NC; ++c)
        for (int q = threadIdx.y; q < 32; q += blockDim.y) {          // read: rows l, columns m_out (contiguous)
            const int l = l0 + q, m = m0 + threadIdx.x;
            const int m_out = (c == 1 || sgn_out < 0) ? -m : m;
            double2 v = make_double2(0.0, 0.0);
            const int am = m < 0 ? -m : m;
            if (l < L && m < L && l >= an && l >= am && !(c == 1 && m == 0 && !fold)) v = coef[(size_t)l * NB + m_out + L - 1];
            tile[c][q][threadIdx.x] = v;
        }
    __syncthreads();
    for (int q = threadIdx.y; q < 32; q += blockDim.y) {              // write: rows m, columns l (contiguous)
        const int m = m0 + q, l = l0 + threadIdx.x;
        if (m >= L || l >= Lp) continue;
        double* g = G + ((size_t)(m - m_end) * Lp + l) * ROWD;
        const double2 sg = SG[(size_t)(l / SHT_TQ) * sgstride + (m - mmin)];
        const double cm = l < L ? scale[l] * C[(size_t)(m - mmin) * Lp + l] : 0.0;
        for (int c = 0; c < NC; ++c) {
            double sgn = 1.0;
            if (c == 1) sgn = fold ? sgn_pow(l - n) : sgn_pow(m);      // fold pass: F_{-m}(pi - theta) = sum_l (-1)^{l-n} f_{l,-m} d^l_{m,n}(theta)
            else if (sgn_out < 0) sgn = sgn_pow(m + n);
            const double2 x = tile[c][threadIdx.x][q];
            g[2 * c] = sgn * cm * x.x; g[2 * c + 1] = sgn * cm * x.y;
        }
        g[2 * NC] = l < L ? (double)(l - m) * (double)(l + m + 1) * sg.y : 0.0;
        g[2 * NC + 1] = sg.x;
    }
}
// pole rings, inverse.  South (theta = pi, Eq. 29): F_{-n}(pi) = sum_l scale(l) f_{l,-n} (-1)^{l-n};  north (theta = 0, Eq. 28,
// MWSS only): F_n(0) = sum_l scale(l) f_{l,n}  (d^l_{mn}(0) = delta_mn, d^l_{mn}(pi) = (-1)^{l+m} delta_{m,-n}).  One block per slab.
__global__ void k_pole_inverse(int L, int north, int NBf, const int* __restrict__ slab_n, const int* __restrict__ cslab,
                               const double2* __restrict__ coef_base, size_t coef_slab, const double* __restrict__ scale,
                               double2* __restrict__ F, size_t F_slab, int ldf, int col) {
    __shared__ double sre[256], sim[256];
    const int slab = blockIdx.x, n = slab_n[slab];
    const double2* coef = coef_base + (size_t)cslab[slab] * coef_slab;
    const int an = n < 0 ? -n : n, NB = 2 * L - 1, m = north ? n : -n;
    double re = 0, im = 0;
    for (int l = an + threadIdx.x; l < L; l += blockDim.x) {
        double2 x = coef[(size_t)l * NB + m + L - 1];
        double s = north ? scale[l] : scale[l] * sgn_pow(l - n);
        re += s * x.x; im += s * x.y;
    }
    sre[threadIdx.x] = re; sim[threadIdx.x] = im;
    __syncthreads();
    for (int k = blockDim.x / 2; k > 0; k >>= 1) {
        if ((int)threadIdx.x < k) { sre[threadIdx.x] += sre[threadIdx.x + k]; sim[threadIdx.x] += sim[threadIdx.x + k]; }
        __syncthreads();
    }
    if (threadIdx.x == 0) F[F_slab * slab + (size_t)(m < 0 ? m + NBf : m) * ldf + col] = make_double2(sre[0], sim[0]);
}
// real signals: rows m < 0 of F from rows m > 0:  F_{-m}(theta) = conj(F_m(theta))
__global__ void k_hermitian_rows(int L, int NB, int ntp, int nth, double2* __restrict__ F) {
    int th = blockIdx.x * blockDim.x + threadIdx.x, m = 1 + blockIdx.y;
    if (th >= nth || m >= L) return;
    double2 v = F[(size_t)m * ntp + th];
    F[(size_t)(NB - m) * ntp + th] = make_double2(v.x, -v.y);
}
__global__ void k_real_to_complex(size_t n, const double* __restrict__ in, double2* __restrict__ out) {
    size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) out[i] = make_double2(in[i], 0.0);
}
__global__ void k_complex_to_real(size_t n, const double2* __restrict__ in, double* __restrict__ out) {
    size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) out[i] = in[i].x;
}

// MW / MWSS forward (ii): extension of F_m(theta_t) to the theta circle of T samples:
//   MW   (mwss = 0): T = 2L-1, theta_t = (2t+1)pi/T, rings t = 0..L-1 given, t = L..2L-2: F_m(theta_t) = (-1)^{m-n} F_m(theta_{2L-2-t})
//   MWSS (mwss = 1): T = 2L,   theta_t = 2 pi t/T,   rings t = 0..L   given, t = L+1..2L-1: F_m(theta_t) = (-1)^{m-n} F_m(theta_{2L-t})
// Rings AT a pole hold one value of a spin-s function (n = -s): at theta = pi only the order m = -n survives (Eq. 29),
// at theta = 0 only m = n (Eq. 28).  The samples of those rings are projected onto that component (F_m := 0 for the other m), which
// makes the transform well defined on arbitrary arrays (R21; include/b200sht.h, s2_forward).
__device__ __forceinline__ double2 mw_ext_value(int L, int n, int mwss, int ldin, const double2* __restrict__ Fa, int m, int t) {
    const int T = mwss ? 2 * L : 2 * L - 1, tpole = mwss ? L : L - 1;
    const int b = m < 0 ? m + T : m;
    double2 v;
    if (t == tpole) { v = Fa[(size_t)b * ldin + t]; if (m != -n) v = make_double2(0.0, 0.0); }
    else if (mwss && t == 0) { v = Fa[(size_t)b * ldin]; if (m != n) v = make_double2(0.0, 0.0); }
    else if (t < tpole) v = Fa[(size_t)b * ldin + t];
    else { v = Fa[(size_t)b * ldin + (2 * tpole - t)]; double s = sgn_pow(m - n); v.x *= s; v.y *= s; }
    return v;
}
// pair = 0: row b of X = the extension of the phi-FFT bin b (order m = b or b - T).  pair != 0: row j = the sum of the extensions of
// the orders 2j-(L-1) and 2j-(L-2) (u_get above), L rows instead of T.
__global__ void k_mw_extend(int L, const int* __restrict__ slab_n, int mwss, int pair, int ldin, int ldout, const double2* __restrict__ Fa_base,
                            size_t Fa_slab, double2* __restrict__ X_base, size_t X_slab) {
    int t = blockIdx.x * blockDim.x + threadIdx.x, b = blockIdx.y;
    const int n = slab_n[blockIdx.z];
    const double2* Fa = Fa_base + Fa_slab * blockIdx.z;
    double2* X = X_base + X_slab * blockIdx.z;
    const int T = mwss ? 2 * L : 2 * L - 1;
    if (t >= T) return;
    double2 v;
    if (pair) {
        const int ma = 2 * b - (L - 1);
        v = mw_ext_value(L, n, mwss, ldin, Fa, ma, t);
        if (ma + 1 <= L - 1) { const double2 w = mw_ext_value(L, n, mwss, ldin, Fa, ma + 1, t); v.x += w.x; v.y += w.y; }
    } else if (mwss && b == L) v = make_double2(0.0, 0.0);           // phi-Nyquist bin of the 2L-point ring FFT: outside the band-limit
    else v = mw_ext_value(L, n, mwss, ldin, Fa, b < L ? b : b - T, t);
    X[(size_t)b * ldout + t] = v;
}
// MW / MWSS forward (iii)->(iv): with Y = FFT_T of the extended samples, F_{mm'} = (1/T) e^{-i m' theta_0} Y[m' mod T] (theta_0 = pi/T
// on MW, 0 on MWSS); Z[m' mod T2] = F_{mm'} e^{+i m' pi/T2} for |m'| <= L-1, zero elsewhere, so that the inverse FFT of length T2 = 4L
// evaluates F_m on the midpoint rings theta'_u = (2u+1) pi/T2 (T2 samples of the circle; u < 2L are the rings in (0, pi)).
__global__ void k_mw_pad_phase(int L, int mwss, int ldin, int ldout, const double2* __restrict__ Y_base, size_t Y_slab,
                               double2* __restrict__ Z_base, size_t Z_slab) {
    int k2 = blockIdx.x * blockDim.x + threadIdx.x, b = blockIdx.y;
    const double2* Y = Y_base + Y_slab * blockIdx.z;
    double2* Z = Z_base + Z_slab * blockIdx.z;
    const int T = mwss ? 2 * L : 2 * L - 1, T2 = ldout;
    if (k2 >= T2) return;
    int mp = k2 < L ? k2 : (k2 > T2 - L ? k2 - T2 : T2);      // |m'| <= L-1, else none
    double2 v = {0.0, 0.0};
    if (mp != T2) {
        double2 y = Y[(size_t)b * ldin + (mp < 0 ? mp + T : mp)];
        double s1 = 0.0, c1 = 1.0, s2, c2;
        if (!mwss) sincospi(-(double)mp / (double)T, &s1, &c1);
        sincospi((double)mp / (double)T2, &s2, &c2);
        double pr = c1 * c2 - s1 * s2, pi_ = c1 * s2 + s1 * c2;
        double inv = 1.0 / (double)T;
        v.x = (y.x * pr - y.y * pi_) * inv; v.y = (y.x * pi_ + y.y * pr) * inv;
    }
    Z[(size_t)b * ldout + k2] = v;
}
// ---- MW inverse through a symmetric intermediate ring set (api.cu `invsym`) ----------------------------------------------
// F_m(theta) of a band-limited signal is a trigonometric polynomial of degree <= L-1 on the theta circle with F_m(2pi - theta) =
// (-1)^{m+s} F_m(theta).  The theta kernel evaluates it on the L midpoint rings vartheta_j = (2j+1)pi/(2L), which are
// symmetric about the equator (north-south fold); these kernels carry it to the MW rings theta_t = (2t+1)pi/(2L-1), exactly:
// extend to the 2L-point circle -> FFT(2L) -> phase and re-bin -> inverse FFT(2L-1) -> keep t = 0..L-1 (t = L-1 is the ring theta = pi).
__global__ void k_sym_extend(int L, int n, int pair, int ldin, const double2* __restrict__ F, double2* __restrict__ X) {
    int j = blockIdx.x * blockDim.x + threadIdx.x, b = blockIdx.y;
    if (j >= 2 * L) return;
    const int T = 2 * L - 1;
    auto ext = [&](int m) {
        const double2* row = F + (size_t)(m < 0 ? m + T : m) * ldin;
        if (j < L) return row[j];
        double2 v = row[2 * L - 1 - j]; const double s = sgn_pow(m - n); v.x *= s; v.y *= s;
        return v;
    };
    double2 v;
    if (pair) {               // row b = orders 2b-(L-1) and 2b-(L-2) summed (u_get above): L rows instead of 2L-1
        const int ma = 2 * b - (L - 1);
        v = ext(ma);
        if (ma + 1 <= L - 1) { const double2 w = ext(ma + 1); v.x += w.x; v.y += w.y; }
    } else v = ext(b < L ? b : b - T);
    X[(size_t)b * 2 * L + j] = v;
}
// paired resampling, last step: X[j][t] (t = 0..2L-2, the MW circle theta_t = (2t+1)pi/(2L-1); mirror of t is 2L-2-t) holds the sum of two
// orders; F[bin(m)][t] = (c[t] + (-1)^{m-n} c[2L-2-t]) / 2 for the rings t = 0..L-1 of the map.
__global__ void k_sym_unpair(int L, int n, int ldout, const double2* __restrict__ X, double2* __restrict__ F) {
    int t = blockIdx.x * blockDim.x + threadIdx.x, b = blockIdx.y;
    if (t >= L) return;
    const int T = 2 * L - 1, m = b < L ? b : b - T;
    const double2* row = X + (size_t)((m + L - 1) >> 1) * T;
    const double2 a = row[t], c = row[T - 1 - t];
    const double s = ((m - n) & 1) ? -0.5 : 0.5;
    F[(size_t)b * ldout + t] = make_double2(fma(s, c.x, 0.5 * a.x), fma(s, c.y, 0.5 * a.y));
}
// Y[b][k] = 2L c_{m'} e^{i m' pi/(2L)} (k = m' mod 2L)  ->  Z[b][m' mod (2L-1)] = c_{m'} e^{i m' pi/(2L-1)}
__global__ void k_sym_rebin(int L, const double2* __restrict__ Y, double2* __restrict__ Z) {
    int k2 = blockIdx.x * blockDim.x + threadIdx.x, b = blockIdx.y;
    const int T = 2 * L - 1;
    if (k2 >= T) return;
    const int mp = k2 < L ? k2 : k2 - T;
    const double2 y = Y[(size_t)b * 2 * L + (mp < 0 ? mp + 2 * L : mp)];
    double s1, c1, s2, c2;
    sincospi(-(double)mp / (double)(2 * L), &s1, &c1);
    sincospi((double)mp / (double)T, &s2, &c2);
    const double pr = c1 * c2 - s1 * s2, pi_ = c1 * s2 + s1 * c2, inv = 1.0 / (double)(2 * L);
    Z[(size_t)b * T + k2] = make_double2((y.x * pr - y.y * pi_) * inv, (y.x * pi_ + y.y * pr) * inv);
}
__global__ void k_rows_head(int ncol, int ldin, int ldout, const double2* __restrict__ in, double2* __restrict__ out) {
    int c = blockIdx.x * blockDim.x + threadIdx.x, b = blockIdx.y;
    if (c < ncol) out[(size_t)b * ldout + c] = in[(size_t)b * ldin + c];
}
// forward split: U[bin][u] (upsampled F_m(theta'_u), or the ring-FFT output on other samplings) -> weighted operand
// tiles W[m-m_end][ntp][NC] of one pass; rings not served by the pass at step m get 0 (peak split, R5).
// fold != 0 (n != 0, symmetric ring set): column 0 = order +m at the ring itself (m >= m_s), column 1 = order -m at the MIRRORED
// ring pi - theta (index nth-1-th), served by the same d-value up to (-1)^{l-n} (applied at the output), for m > m_s.
__global__ void k_weight_split(int L, int NBin, int ldin, int pair, int nth, int ntp, int NC, const double* __restrict__ wq,
                               const double2* __restrict__ U_base, size_t U_slab, const ThetaPass* __restrict__ passes, int th_lo, int th_hi) {
    // one launch serves all passes of a kernel mode: grid.z = pass (its operand rows start one row into ThetaPass::in)
    const ThetaPass P = passes[blockIdx.z];
    const int n = P.sgn_out > 0 ? P.n : -P.n, sgn_out = P.sgn_out, m_end = P.m_end, fold = P.fold;
    const int* __restrict__ m_lo = P.m_lo;
    const double2* U = U_base + U_slab * P.slab;
    double2* W = reinterpret_cast<double2*>(const_cast<double*>(P.in)) + (size_t)ntp * NC;
    if (m_end + (int)blockIdx.y >= L) return;
    int th = blockIdx.x * blockDim.x + threadIdx.x;
    int m = m_end + blockIdx.y;
    if (th >= ntp) return;
    for (int c = 0; c < NC; ++c) {
        double2 v = {0.0, 0.0};
        bool ok = th < nth && (m < L) && (m > -L) && th >= th_lo && th < th_hi;
        if (fold) { if (ok) ok = c == 0 ? m >= m_lo[th] : m > m_lo[th]; }
        else {
            ok = ok && !(c == 1 && m == 0);
            if (ok && m_lo) ok = m >= m_lo[th];
        }
        if (ok) {
            int m_out = (c == 1 || sgn_out < 0) ? -m : m;
            const int ts = (fold && c == 1) ? nth - 1 - th : th;
            double s = wq[ts];
            if (!fold) {
                if (c == 1) s *= sgn_pow(m);
                else if (sgn_out < 0) s *= sgn_pow(m + n);
            }
            double2 x = u_get(U, ldin, NBin, pair, L, n, m_out, ts);
            v.x = s * x.x; v.y = s * x.y;
        }
        W[((size_t)(m - m_end) * ntp + th) * NC + c] = v;
    }
}
// forward split for n = 0 on a ring set symmetric about the equator (theta_kernels.cu FOLD): only the nth northern rings are
// recursed.  W[m][ntp][2][NC]: set 0 = E = q (F_m(theta) + F_m(pi - theta)), set 1 = O = q (F_m(theta) - F_m(pi - theta)); the mirror of
// ring th is nfull-1-th (the equator ring of HEALPix is its own mirror: E = q F_m, O = 0).  Column c = 1 is order -m with (-1)^m.
__global__ void k_weight_split_fold0(int L, int NBin, int ldin, int pair, int nth, int ntp, int nfull, int NC, int m_end,
                                     const double* __restrict__ wq, const double2* __restrict__ U, double2* __restrict__ W, int th_lo, int th_hi) {
    int th = blockIdx.x * blockDim.x + threadIdx.x;
    int m = m_end + blockIdx.y;
    if (th >= ntp) return;
    for (int c = 0; c < NC; ++c) {
        double2 e = {0.0, 0.0}, o = {0.0, 0.0};
        if (th < nth && !(c == 1 && m == 0) && m < L && m > -L && th >= th_lo && th < th_hi) {
            const int m_out = c == 1 ? -m : m, tm = nfull - 1 - th;
            double s = wq[th];
            if (c == 1) s *= sgn_pow(m);
            const double2 a = u_get(U, ldin, NBin, pair, L, 0, m_out, th);
            double2 b = {0.0, 0.0};
            if (tm != th) b = u_get(U, ldin, NBin, pair, L, 0, m_out, tm);
            e.x = s * (a.x + b.x); e.y = s * (a.y + b.y);
            if (tm != th) { o.x = s * (a.x - b.x); o.y = s * (a.y - b.y); }
        }
        double2* w = W + ((size_t)(m - m_end) * ntp + th) * 2 * NC;
        w[c] = e; w[NC + c] = o;
    }
}
// pole rings, forward.  South (theta = pi, Eq. 29): H[-n+L-1][l] += (-1)^{l-n} w U_{-n}(pi);  north (theta = 0, Eq. 28): H[n+L-1][l] += w U_n(0).
// `col` is the ring's column of U (may be -1 when U points at the first regular ring and the north pole precedes it).
__global__ void k_pole_forward(int L, int Lp, int n, int north, int NBin, int ldin, int col, double w, const double2* __restrict__ U,
                               double2* __restrict__ H) {
    int l = blockIdx.x * blockDim.x + threadIdx.x;
    const int an = n < 0 ? -n : n;
    if (l >= L || l < an) return;
    int mo = north ? n : -n;
    double2 x = U[(ptrdiff_t)(mo < 0 ? mo + NBin : mo) * ldin + col];
    double s = north ? w : w * sgn_pow(l - n);
    double2* h = H + (size_t)(mo + L - 1) * Lp + l;
    h->x += s * x.x; h->y += s * x.y;
}
// forward finalize: H[m+L-1][Lp] -> coef[l][m+L-1] = scale(l) * H on the support, 0 elsewhere; real: fill m<0.
__global__ void k_finalize_forward(int L, int Lp, const int* __restrict__ slab_n, const int* __restrict__ cslab, int real,
                                   const double* __restrict__ scale, const double2* __restrict__ H_base, size_t H_slab,
                                   double2* __restrict__ coef_base, size_t coef_slab) {
    __shared__ double2 tile[32][33];
    const int n = slab_n[blockIdx.z];
    const double2* H = H_base + H_slab * blockIdx.z;
    double2* coef = coef_base + (size_t)cslab[blockIdx.z] * coef_slab;
    const int NB = 2 * L - 1, an = n < 0 ? -n : n;
    int mi0 = blockIdx.x * 32, l0 = blockIdx.y * 32;
    for (int r = threadIdx.y; r < 32; r += blockDim.y) {      // read H rows (mi), coalesced along l
        int mi = mi0 + r, l = l0 + threadIdx.x;
        double2 v = {0.0, 0.0};
        if (mi < NB && l < L) {
            int m = mi - (L - 1), am = m < 0 ? -m : m;
            if (l >= an && l >= am) {
                if (real && m < 0) { double2 h = H[(size_t)(-m + L - 1) * Lp + l]; double s = scale[l] * sgn_pow(m); v.x = s * h.x; v.y = -s * h.y; }
                else { double2 h = H[(size_t)mi * Lp + l]; v.x = scale[l] * h.x; v.y = scale[l] * h.y; }
            }
        }
        tile[r][threadIdx.x] = v;
    }
    __syncthreads();
    for (int r = threadIdx.y; r < 32; r += blockDim.y) {      // write coef rows (l), coalesced along mi
        int l = l0 + r, mi = mi0 + threadIdx.x;
        if (l < L && mi < NB) coef[(size_t)l * NB + mi] = tile[threadIdx.x][r];
    }
}
// 32 x 32 tile transpose of nslab matrices: out[slab][c][r] = in[slab][r][c] (r < nrow, c < ncol; row lengths ldin / ldout)
__global__ void k_transpose_slabs(int nrow, int ncol, int ldin, int ldout, const double2* __restrict__ in, size_t in_slab,
                                  double2* __restrict__ out, size_t out_slab) {
    __shared__ double2 tile[32][33];
    in += in_slab * blockIdx.z; out += out_slab * blockIdx.z;
    const int r0 = blockIdx.y * 32, c0 = blockIdx.x * 32;
    for (int q = threadIdx.y; q < 32; q += blockDim.y) {
        const int r = r0 + q, c = c0 + threadIdx.x;
        tile[q][threadIdx.x] = (r < nrow && c < ncol) ? in[(size_t)r * ldin + c] : make_double2(0.0, 0.0);
    }
    __syncthreads();
    for (int q = threadIdx.y; q < 32; q += blockDim.y) {
        const int c = c0 + q, r = r0 + threadIdx.x;
        if (c < ncol && r < nrow) out[(size_t)c * ldout + r] = tile[threadIdx.x][q];
    }
}
// generic strided row copy used by the theta-stage entry points: dst[r][c] = src[map(r)][c]
__global__ void k_rows_bin_to_mi(int L, int NB, int ncol, int ldsrc, int lddst, int to_mi, const double2* __restrict__ src,
                                 double2* __restrict__ dst) {
    int c = blockIdx.x * blockDim.x + threadIdx.x, r = blockIdx.y;
    if (c >= ncol) return;
    int m = r - (L - 1);
    int b = m < 0 ? m + NB : m;
    if (to_mi) dst[(size_t)r * lddst + c] = src[(size_t)b * ldsrc + c];
    else dst[(size_t)b * lddst + c] = src[(size_t)r * ldsrc + c];
}
// SO(3): coefficient slabs are stored in n order (n+N-1); internal slabs are in gamma-FFT bin order (n mod 2N-1)
__global__ void k_scale_copy(size_t n, double s, const double2* __restrict__ in, double2* __restrict__ out) {
    size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) out[i] = make_double2(s * in[i].x, s * in[i].y);
}

// ---- adjoint transforms (Sec. 5.3): conjugate transposes of the staging steps above -------------------------------
// F[row][c] *= w[c]: the diagonal operator Q of Eq. 52 on the rings of the map (direct-quadrature samplings)
// out[l][c] = sgn * d[l] * in[l][c]  (row-wise l-scaling of a coefficient slab; SO(3) adjoints)
__global__ void k_scale_rows(int nrow, int ncol, double sgn, const double* __restrict__ d, const double2* __restrict__ in, double2* __restrict__ out) {
    int c = blockIdx.x * blockDim.x + threadIdx.x, l = blockIdx.y;
    if (c >= ncol) return;
    const double s = sgn * d[l];
    const double2 v = in[(size_t)l * ncol + c];
    out[(size_t)l * ncol + c] = make_double2(s * v.x, s * v.y);
}
__global__ void k_scale_cols(int ncol, int ld, const double* __restrict__ w, double2* __restrict__ F) {
    int c = blockIdx.x * blockDim.x + threadIdx.x, r = blockIdx.y;
    if (c >= ncol) return;
    double2 v = F[(size_t)r * ld + c];
    const double s = w[c];
    F[(size_t)r * ld + c] = make_double2(s * v.x, s * v.y);
}
// Adjoint of "weights, restriction to u < 2L": Z[bin(m)][u] = q_u Fq[binq(m)][u] for u < 2L, 0 for 2L <= u < T2 = 4L.  Fq has NBq = 2L-1
// bins (the helper plan's rows), Z has NB bins; on MWSS the phi-Nyquist bin b = L carries nothing.
__global__ void k_adj_weight_pad(int L, int NBq, int ldq, const double2* __restrict__ Fq, const double* __restrict__ wq, int NB, int T2,
                                 double2* __restrict__ Z) {
    int u = blockIdx.x * blockDim.x + threadIdx.x, b = blockIdx.y;
    if (u >= T2) return;
    double2 v = make_double2(0.0, 0.0);
    const int m = b < L ? b : b - NB;
    if (u < 2 * L && m > -L) {
        const double2 x = Fq[(size_t)(m < 0 ? m + NBq : m) * ldq + u];
        v = make_double2(wq[u] * x.x, wq[u] * x.y);
    }
    Z[(size_t)b * T2 + u] = v;
}
// Adjoint of k_mw_pad_phase: X[b][m' mod T] = (1/T) e^{+i m' theta_0} e^{-i m' pi/T2} Zf[b][m' mod T2] for |m'| <= L-1, 0 elsewhere
__global__ void k_adj_trunc_phase(int L, int mwss, int T2, const double2* __restrict__ Zf, double2* __restrict__ X) {
    int k = blockIdx.x * blockDim.x + threadIdx.x, b = blockIdx.y;
    const int T = mwss ? 2 * L : 2 * L - 1;
    if (k >= T) return;
    const int mp = k < L ? k : k - T;
    double2 v = make_double2(0.0, 0.0);
    if (mp > -L) {
        const double2 y = Zf[(size_t)b * T2 + (mp < 0 ? mp + T2 : mp)];
        double s1 = 0.0, c1 = 1.0, s2, c2;
        if (!mwss) sincospi((double)mp / (double)T, &s1, &c1);
        sincospi(-(double)mp / (double)T2, &s2, &c2);
        const double pr = c1 * c2 - s1 * s2, pi_ = c1 * s2 + s1 * c2, inv = 1.0 / (double)T;
        v = make_double2((y.x * pr - y.y * pi_) * inv, (y.x * pi_ + y.y * pr) * inv);
    }
    X[(size_t)b * T + k] = v;
}
// Adjoint of k_mw_extend: F[b][t] = X[b][t] + (-1)^{m-n} X[b][2 t_pole - t] on the regular rings; the pole rings keep X only for the one
// order a spin function can hold there (the projection is diagonal, hence self-adjoint); the MWSS phi-Nyquist bin is zero.
__global__ void k_adj_fold(int L, int n, int mwss, int nrmap, int ldf, const double2* __restrict__ X, double2* __restrict__ F) {
    int t = blockIdx.x * blockDim.x + threadIdx.x, b = blockIdx.y;
    const int T = mwss ? 2 * L : 2 * L - 1, tpole = mwss ? L : L - 1;
    if (t >= nrmap) return;
    const int m = b < L ? b : b - T;
    const double2* x = X + (size_t)b * T;
    double2 v = make_double2(0.0, 0.0);
    if (mwss && b == L) { }
    else if (t == tpole) { if (m == -n) v = x[t]; }
    else if (mwss && t == 0) { if (m == n) v = x[0]; }
    else { const double2 r = x[2 * tpole - t]; const double s = sgn_pow(m - n); v = make_double2(x[t].x + s * r.x, x[t].y + s * r.y); }
    F[(size_t)b * ldf + t] = v;
}

// ---- HEALPix iterative refinement: residual and update, plain vector kernels
__global__ void k_vec_sub(size_t n, const double* __restrict__ a, const double* __restrict__ b, double* __restrict__ out) {
    size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) out[i] = a[i] - b[i];
}
__global__ void k_vec_add(size_t n, const double* __restrict__ x, double* __restrict__ y) {
    size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) y[i] += x[i];
}

// ---- batched path (theta_mma.cu; operand layouts in internal.h) ----------------------------------------------------
// Complex column j = cg*16 + jc of a pass belongs to map b = j / NC and, with NC = 2 (spin 0 complex), to order +m
// (c = 0) or -m (c = 1); columns j >= B*NC are zero padding.
// inverse prep: coef[b][l][NB] -> Gb[cg][m-m_end][Lp][36].  Block = 16 degrees x 8 orders x one column group.
__global__ void k_prep_inverse_batch(int L, int Lp, int NC, int B, int n, int sgn_out, int m_end, int mmin,
                                     const double2* __restrict__ coef, const double* __restrict__ scale, const double* __restrict__ C,
                                     const double2* __restrict__ SG, int sgstride, double* __restrict__ Gb, size_t cg_stride) {
    __shared__ double2 tile[16][16][9];
    const int NB = 2 * L - 1, an = n < 0 ? -n : n, cg = blockIdx.z;
    const int l0 = blockIdx.x * 16, m0 = m_end + blockIdx.y * 8;
    const int tx = threadIdx.x & 7, ty = threadIdx.x >> 3;
    for (int jc = 0; jc < 16; ++jc) {
        const int j = cg * 16 + jc, b = j / NC, c = j % NC;
        const int l = l0 + ty, m = m0 + tx, am = m < 0 ? -m : m;
        const int m_out = (c == 1 || sgn_out < 0) ? -m : m;
        double2 v = make_double2(0.0, 0.0);
        if (b < B && l < L && m < L && l >= an && l >= am && !(c == 1 && m == 0)) {
            v = coef[((size_t)b * L + l) * NB + m_out + L - 1];
            double sgn = 1.0;
            if (c == 1) sgn = sgn_pow(m);
            else if (sgn_out < 0) sgn = sgn_pow(m + n);
            const double cm = sgn * scale[l] * C[(size_t)(m - mmin) * Lp + l];
            v.x *= cm; v.y *= cm;
        }
        tile[ty][jc][tx] = v;
    }
    __syncthreads();
    for (int mi = 0; mi < 8; ++mi) {
        const int m = m0 + mi;
        if (m >= L) break;
        double* g = Gb + (size_t)cg * cg_stride + ((size_t)(m - m_end) * Lp + l0) * SHT_MMA_ROW;
        for (int idx = threadIdx.x; idx < 16 * SHT_MMA_ROW; idx += blockDim.x) {
            const int li = idx / SHT_MMA_ROW, col = idx % SHT_MMA_ROW, l = l0 + li;
            double v = 0.0;
            if (col < SHT_MMA_NCOL) { const double2 t = tile[li][col >> 1][mi]; v = (col & 1) ? t.y : t.x; }
            else if (col == SHT_MMA_NCOL) v = l < L ? (double)(l - m) * (double)(l + m + 1) * SG[(size_t)(l / SHT_TQ) * sgstride + (m - mmin)].y : 0.0;
            else if (col == SHT_MMA_NCOL + 1) v = SG[(size_t)(l / SHT_TQ) * sgstride + (m - mmin)].x;
            g[idx] = v;
        }
    }
}
// forward split: U[b][bin][ldu] -> Wb[cg][m-m_end][ntp][36] (weighted, masked by the peak split; [32] = lambda_m(theta)).
// Block = 32 rings x one order x one column group.
__global__ void k_weight_split_batch(int L, int NBin, int ldin, int pair, size_t U_slab, int nth, int ntp, int NC, int B, int n, int sgn_out,
                                     int m_end, int fold, const int* __restrict__ m_lo, const double* __restrict__ wq,
                                     const double* __restrict__ lam, const double2* __restrict__ U, double* __restrict__ Wb,
                                     size_t cg_stride) {
    __shared__ double2 tile[32][17];
    const int cg = blockIdx.z, m = m_end + blockIdx.y, t0 = blockIdx.x * 32;
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5, th = t0 + tx;
    for (int jc = ty; jc < 16; jc += 4) {
        const int j = cg * 16 + jc, b = j / NC, c = j % NC;
        double2 v = make_double2(0.0, 0.0);
        bool ok = b < B && th < nth && m < L && m > -L;
        if (fold) { if (ok) ok = c == 0 ? m >= m_lo[th] : m > m_lo[th]; }
        else {
            ok = ok && !(c == 1 && m == 0);
            if (ok && m_lo) ok = m >= m_lo[th];
        }
        if (ok) {
            const int m_out = (c == 1 || sgn_out < 0) ? -m : m;
            const int ts = (fold && c == 1) ? nth - 1 - th : th;
            double s = wq[ts];
            if (!fold) {
                if (c == 1) s *= sgn_pow(m);
                else if (sgn_out < 0) s *= sgn_pow(m + n);
            }
            const double2 x = u_get(U + (size_t)b * U_slab, ldin, NBin, pair, L, n, m_out, ts);      // (n = the slab's second index)
            v.x = s * x.x; v.y = s * x.y;
        }
        tile[tx][jc] = v;
    }
    __syncthreads();
    double* g = Wb + (size_t)cg * cg_stride + ((size_t)(m - m_end) * ntp + t0) * SHT_MMA_ROW;
    for (int idx = threadIdx.x; idx < 32 * SHT_MMA_ROW; idx += blockDim.x) {
        const int ti = idx / SHT_MMA_ROW, col = idx % SHT_MMA_ROW;
        double v = 0.0;
        if (col < SHT_MMA_NCOL) { const double2 t = tile[ti][col >> 1]; v = (col & 1) ? t.y : t.x; }
        else if (col == SHT_MMA_NCOL) v = lam[(size_t)(m - m_end + 1) * ntp + t0 + ti];
        g[idx] = v;
    }
}
// forward split of the n = 0 fold (theta_mma.cu FOLD): Wb[cg][m-m_end][ntp north][68] = {32 columns E, 32 columns O, lambda, pad};
// E = q (F_m(theta) + F_m(pi - theta)), O = q (F_m(theta) - F_m(pi - theta)), mirror ring index nfull-1-th.
__global__ void k_weight_split_batch_fold0(int L, int NBin, int ldin, int pair, size_t U_slab, int nth, int ntp, int nfull, int NC, int B, int m_end,
                                           const double* __restrict__ wq, const double* __restrict__ lam,
                                           const double2* __restrict__ U, double* __restrict__ Wb, size_t cg_stride) {
    __shared__ double2 tile[2][32][17];
    const int cg = blockIdx.z, m = m_end + blockIdx.y, t0 = blockIdx.x * 32;
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5, th = t0 + tx;
    for (int jc = ty; jc < 16; jc += 4) {
        const int j = cg * 16 + jc, b = j / NC, c = j % NC;
        double2 e = make_double2(0.0, 0.0), o = make_double2(0.0, 0.0);
        if (b < B && th < nth && !(c == 1 && m == 0) && m < L && m > -L) {
            const int m_out = c == 1 ? -m : m, tm = nfull - 1 - th;
            const double2* Ub = U + (size_t)b * U_slab;
            double s = wq[th];
            if (c == 1) s *= sgn_pow(m);
            const double2 a = u_get(Ub, ldin, NBin, pair, L, 0, m_out, th);
            double2 v = make_double2(0.0, 0.0);
            if (tm != th) v = u_get(Ub, ldin, NBin, pair, L, 0, m_out, tm);
            e.x = s * (a.x + v.x); e.y = s * (a.y + v.y);
            if (tm != th) { o.x = s * (a.x - v.x); o.y = s * (a.y - v.y); }
        }
        tile[0][tx][jc] = e; tile[1][tx][jc] = o;
    }
    __syncthreads();
    double* g = Wb + (size_t)cg * cg_stride + ((size_t)(m - m_end) * ntp + t0) * SHT_MMA_ROWF;
    for (int idx = threadIdx.x; idx < 32 * SHT_MMA_ROWF; idx += blockDim.x) {
        const int ti = idx / SHT_MMA_ROWF, col = idx % SHT_MMA_ROWF;
        double v = 0.0;
        if (col < 2 * SHT_MMA_NCOL) { const int cc = col % SHT_MMA_NCOL; const double2 t = tile[col / SHT_MMA_NCOL][ti][cc >> 1]; v = (cc & 1) ? t.y : t.x; }
        else if (col == 2 * SHT_MMA_NCOL) v = lam[(size_t)(m - m_end + 1) * ntp + t0 + ti];
        g[idx] = v;
    }
}
// results: Ob[cg][m-m_end][Mp][32] -> out[b][row(m_out)][ld] += factor * value, complex.  fwd = 0: rows are phi-FFT bins
// (m_out mod NB) of F, columns rings; fwd = 1: rows m_out+L-1 of H, columns degrees, factor c_m(l) (internal.h).
__global__ void k_unpack_batch(int L, int Lp, int Mp, int mlim, int NC, int B, int n, int sgn_out, int m_end, int mmin, int fwd, int fold,
                               const double* __restrict__ C, const double* __restrict__ Ob, size_t cg_stride,
                               double2* __restrict__ out, size_t out_slab, int ld) {
    __shared__ double tile[32][33];
    const int NB = 2 * L - 1, an = n < 0 ? -n : n;
    const int cg = blockIdx.z, m = m_end + blockIdx.y, i0 = blockIdx.x * 32;
    const double* src = Ob + (size_t)cg * cg_stride + ((size_t)(m - m_end) * Mp + i0) * SHT_MMA_NCOL;
    for (int idx = threadIdx.x; idx < 32 * SHT_MMA_NCOL; idx += blockDim.x) tile[idx / SHT_MMA_NCOL][idx % SHT_MMA_NCOL] = src[idx];
    __syncthreads();
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5, mi = i0 + tx, am = m < 0 ? -m : m;
    if (mi >= mlim || m >= L || m <= -L) return;
    double fac = 1.0;
    if (fwd) {
        if (mi < an || mi < am) return;
        fac = C[(size_t)(m - mmin) * Lp + mi];
    }
    for (int jc = ty; jc < 16; jc += 4) {
        const int j = cg * 16 + jc, b = j / NC, c = j % NC;
        if (b >= B || (c == 1 && m == 0 && !fold)) continue;
        const int m_out = (c == 1 || sgn_out < 0) ? -m : m;
        const int row = fwd ? m_out + L - 1 : (m_out < 0 ? m_out + NB : m_out);
        double2* o = out + (size_t)b * out_slab + (size_t)row * ld + mi;
        const double f2 = (fold && c == 1 && ((mi - n) & 1)) ? -fac : fac;       // (-1)^{l-n} on the mirrored-ring column
        if (fold && am <= an) {      // rows |m_out| <= |n| receive step m (own ring) and step -m (mirrored ring) of the same launch
            atomicAdd(&o->x, f2 * tile[tx][2 * jc]); atomicAdd(&o->y, f2 * tile[tx][2 * jc + 1]);
            continue;
        }
        double2 v = *o;
        v.x += f2 * tile[tx][2 * jc]; v.y += f2 * tile[tx][2 * jc + 1];
        *o = v;
    }
}

// ---- fp32 variant (theta_f32.cu) ----------------------------------------------------------------------------------------
// recursion coefficients of Eq. 25-26 in the paper's own form, fp32, duplicated for the packed arithmetic of theta_f32.cu:
// AB[m][l] = {A, A, -B, -B}, A = a_{m-1}(l), B = a_{m-1}(l)/a_m(l), a_m = 2/sqrt((l-m)(l+m+1))
__global__ void k_ab32(int L, int Lp, float4* __restrict__ AB) {
    int l = blockIdx.x * blockDim.x + threadIdx.x, m = blockIdx.y;
    if (l >= Lp) return;
    float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
    if (l < L && m >= 1 && l >= m) {
        const double p = (double)(l - m + 1) * (double)(l + m);
        v.x = v.y = (float)(2.0 / sqrt(p));
        v.z = v.w = -(float)sqrt((double)(l - m) * (double)(l + m + 1) / p);
    }
    AB[(size_t)m * Lp + l] = v;
}
// fp64 windowed start values (stride 2^480, internal.h) -> fp32 windowed ones (stride 2^48, top 2^-64)
__global__ void k_start32(size_t n, const double* __restrict__ v64, const uint8_t* __restrict__ k64, float* __restrict__ v32,
                          uint16_t* __restrict__ k16) {
    size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const double v = v64[i];
    float o = 0.f; int k = 0;
    if (v != 0.0) {
        int ex; (void)frexp(v, &ex);                       // |v| = f 2^ex, f in [0.5, 1)
        const long e = (long)ex - (long)SHT_SWIN * k64[i];  // true value = f 2^e
        if (e > -64) k = 0; else k = (int)((-64 - e) / 48 + 1);
        if (k <= 65535) o = (float)ldexp(v, (int)(48L * k - (long)SHT_SWIN * k64[i]));
        else k = 0;
    }
    v32[i] = o; k16[i] = (uint16_t)k;
}
// inverse operands: G32[m][Lp][NC] = scale(l) f_{l,+m} and, for NC = 2, (-1)^m scale(l) f_{l,-m} (32 x 32 transpose, coef is l-major)
__global__ void k_prep_inverse_f32(int L, int Lp, int NC, const double2* __restrict__ coef, const double* __restrict__ scale,
                                   float4* __restrict__ G) {
    __shared__ double2 tile[2][32][33];
    const int NB = 2 * L - 1, l0 = blockIdx.x * 32, m0 = blockIdx.y * 32;
    for (int c = 0; c < NC; ++c)
        for (int q = threadIdx.y; q < 32; q += blockDim.y) {
            const int l = l0 + q, m = m0 + threadIdx.x;
            double2 v = make_double2(0.0, 0.0);
            if (l < L && m < L && l >= m && !(c == 1 && m == 0)) v = coef[(size_t)l * NB + (c == 1 ? -m : m) + L - 1];
            tile[c][q][threadIdx.x] = v;
        }
    __syncthreads();
    for (int q = threadIdx.y; q < 32; q += blockDim.y) {
        const int m = m0 + q, l = l0 + threadIdx.x;
        if (m >= L || l >= Lp) continue;
        const double sc = l < L ? scale[l] : 0.0;
        for (int c = 0; c < NC; ++c) {
            const double sg = (c == 1 && (m & 1)) ? -sc : sc;
            const double2 x = tile[c][threadIdx.x][q];
            const float gx = (float)(sg * x.x), gy = (float)(sg * x.y);
            G[((size_t)m * Lp + l) * NC + c] = make_float4(gx, gx, gy, gy);       // duplicated for the packed arithmetic
        }
    }
}
// forward operands of the fp32 kernels, laid out for packed (two rings per instruction) arithmetic: per order m and ring PAIR
// (2p, 2p+1), NSET operand sets of 2 NC components {Re +m, Im +m[, Re -m, Im -m]}, each a float2 = (ring 2p, ring 2p+1):
//   W32[m][ntp/2][NSET][2 NC] float2.     value = q(theta) F_{+m}(theta) and, for NC = 2, (-1)^m q(theta) F_{-m}(theta)
__device__ __forceinline__ void w32_store(float* __restrict__ W, int m, int ntp, int th, int NSET, int set, int NC, int c, float2 v) {
    float* w = W + ((((size_t)m * (ntp / 2) + (th >> 1)) * NSET + set) * 2 * NC + 2 * c) * 2 + (th & 1);
    w[0] = v.x; w[2] = v.y;
}
__global__ void k_weight_split_f32(int L, int NBin, int ldin, int pair, int nth, int ntp, int NC, const double* __restrict__ wq,
                                   const double2* __restrict__ U, float* __restrict__ W) {
    int th = blockIdx.x * blockDim.x + threadIdx.x, m = blockIdx.y;
    if (th >= ntp) return;
    for (int c = 0; c < NC; ++c) {
        float2 v = make_float2(0.f, 0.f);
        if (th < nth && !(c == 1 && m == 0)) {
            const int m_out = c == 1 ? -m : m;
            const double s = (c == 1 && (m & 1)) ? -wq[th] : wq[th];
            const double2 x = u_get(U, ldin, NBin, pair, L, 0, m_out, th);
            v = make_float2((float)(s * x.x), (float)(s * x.y));
        }
        w32_store(W, m, ntp, th, 1, 0, NC, c, v);
    }
}
// the same for the north-south fold: NSET = 2, set 0 = E = q (F(theta) + F(pi - theta)), set 1 = O = q (F(theta) - F(pi - theta)), northern rings
__global__ void k_weight_split_f32_fold0(int L, int NBin, int ldin, int pair, int nth, int ntp, int nfull, int NC, const double* __restrict__ wq,
                                         const double2* __restrict__ U, float* __restrict__ W) {
    int th = blockIdx.x * blockDim.x + threadIdx.x, m = blockIdx.y;
    if (th >= ntp) return;
    for (int c = 0; c < NC; ++c) {
        float2 e = make_float2(0.f, 0.f), o = make_float2(0.f, 0.f);
        if (th < nth && !(c == 1 && m == 0)) {
            const int m_out = c == 1 ? -m : m, tm = nfull - 1 - th;
            const double s = (c == 1 && (m & 1)) ? -wq[th] : wq[th];
            const double2 a = u_get(U, ldin, NBin, pair, L, 0, m_out, th);
            double2 b = make_double2(0.0, 0.0);
            if (tm != th) b = u_get(U, ldin, NBin, pair, L, 0, m_out, tm);
            e = make_float2((float)(s * (a.x + b.x)), (float)(s * (a.y + b.y)));
            if (tm != th) o = make_float2((float)(s * (a.x - b.x)), (float)(s * (a.y - b.y)));
        }
        w32_store(W, m, ntp, th, 2, 0, NC, c, e);
        w32_store(W, m, ntp, th, 2, 1, NC, c, o);
    }
}
__global__ void k_c64_to_c128(size_t n, const float* __restrict__ in, double* __restrict__ out) {
    size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) out[i] = (double)in[i];
}
__global__ void k_c128_to_c64(size_t n, const double* __restrict__ in, float* __restrict__ out) {
    size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) out[i] = (float)in[i];
}

inline unsigned cdiv(size_t a, size_t b) { return (unsigned)((a + b - 1) / b); }

}  // namespace

#define LAUNCHED() do { count_launch(); cudaError_t e_ = cudaGetLastError(); if (e_ != cudaSuccess) return e_; } while (0)

cudaError_t st_start_values(int L, int n, int nth, int ntp, const double* c2hi, const double* c2lo, const double* s2hi,
                            const double* s2lo, const double* rhi, const double* rlo, double* st_val, uint8_t* st_k, int* range_flag,
                            cudaStream_t st) {
    if (nth <= 0) return cudaSuccess;
    k_start_values<<<cdiv(nth, 64), 64, 0, st>>>(L, n, nth, ntp, c2hi, c2lo, s2hi, s2lo, rhi, rlo, st_val, st_k, range_flag);
    LAUNCHED(); return cudaSuccess;
}
cudaError_t st_kexp(int nrows, int kstride, int kmin, int8_t* kexp, cudaStream_t st) {
    k_kexp<<<cdiv(nrows, 32), 32, 0, st>>>(nrows, kstride, kmin, kexp);
    LAUNCHED(); return cudaSuccess;
}
cudaError_t st_rsq(int n, double* rsq, cudaStream_t st) {
    k_rsq<<<cdiv(n, 256), 256, 0, st>>>(n, rsq);
    LAUNCHED(); return cudaSuccess;
}
cudaError_t st_mid_weights(int L, int count, double qphi, double* w, cudaStream_t st) {
    k_mid_weights<<<cdiv(count, 128), 128, 0, st>>>(L, count, qphi, w);
    LAUNCHED(); return cudaSuccess;
}
cudaError_t st_mw_weights(int Lq, double qphi, double* w, cudaStream_t st) {
    k_mw_weights<<<cdiv(Lq, 128), 128, 0, st>>>(Lq, qphi, w);
    LAUNCHED(); return cudaSuccess;
}
cudaError_t st_prep_inverse(int L, int Lp, int NC, int mmin, int npass, const double2* coef, size_t coef_slab, const int* cslab,
                            const double* scale, const double* C, const double2* SG, int sgstride, const ThetaPass* passes, cudaStream_t st) {
    if (npass == 0) return cudaSuccess;
    dim3 grid(cdiv(Lp, 32), cdiv(L - mmin - 1, 32), npass), block(32, 8);
    k_prep_inverse<<<grid, block, 0, st>>>(L, Lp, NC, mmin, coef, coef_slab, cslab, scale, C, SG, sgstride, passes);
    count_bytes(npass * (16.0 * NC * (double)L * L / 2 + 8.0 * (2 * NC + 2) * (double)L * Lp)); LAUNCHED(); return cudaSuccess;
}
cudaError_t st_ctab(int L, int Lp, int mmin, int kstride, int kmin, const int8_t* kexp, const double* rsq, double* C, cudaStream_t st) {
    k_ctab<<<cdiv(Lp, 64), 64, 0, st>>>(L, Lp, mmin, kstride, kmin, kexp, rsq, C);
    LAUNCHED(); return cudaSuccess;
}
cudaError_t st_sgtab(int nrows, int ncol, int mmin, int kstride, int kmin, const int8_t* kexp, double2* SG, cudaStream_t st) {
    k_sgtab<<<dim3(cdiv(ncol, 128), nrows), 128, 0, st>>>(nrows, ncol, mmin, kstride, kmin, kexp, SG);
    LAUNCHED(); return cudaSuccess;
}
cudaError_t st_lamtab(int n, int nth, int ntp, int m_end, int nrows, const double* csc, const double* tau, const double* sig, double* lam,
                      cudaStream_t st) {
    k_lamtab<<<dim3(cdiv(ntp, 128), nrows), 128, 0, st>>>(n, nth, ntp, m_end, csc, tau, sig, lam);
    LAUNCHED(); return cudaSuccess;
}
cudaError_t st_pole_inverse(int L, int north, int NBf, int nslab, const int* slab_n, const int* cslab, const double2* coef, size_t coef_slab,
                            const double* scale, double2* F, size_t F_slab, int ldf, int col, cudaStream_t st) {
    k_pole_inverse<<<nslab, 256, 0, st>>>(L, north, NBf, slab_n, cslab, coef, coef_slab, scale, F, F_slab, ldf, col);
    count_bytes(16.0 * L * nslab); LAUNCHED(); return cudaSuccess;
}
cudaError_t st_hermitian_rows(int L, int NB, int ntp, int nth, double2* F, cudaStream_t st) {
    if (L < 2) return cudaSuccess;
    dim3 grid(cdiv(nth, 128), L - 1);
    k_hermitian_rows<<<grid, 128, 0, st>>>(L, NB, ntp, nth, F);
    count_bytes(32.0 * (double)(L - 1) * nth); LAUNCHED(); return cudaSuccess;
}
cudaError_t st_real_to_complex(size_t n, const double* in, double2* out, cudaStream_t st) {
    k_real_to_complex<<<cdiv(n, 256), 256, 0, st>>>(n, in, out);
    count_bytes(24.0 * (double)n); LAUNCHED(); return cudaSuccess;
}
cudaError_t st_complex_to_real(size_t n, const double2* in, double* out, cudaStream_t st) {
    k_complex_to_real<<<cdiv(n, 256), 256, 0, st>>>(n, in, out);
    count_bytes(24.0 * (double)n); LAUNCHED(); return cudaSuccess;
}
cudaError_t st_mw_extend(int L, int nslab, const int* slab_n, int mwss, int pair, int ldin, int ldout, const double2* Fa, size_t Fa_slab,
                         double2* X, size_t X_slab, cudaStream_t st) {
    const int T = mwss ? 2 * L : 2 * L - 1, rows = pair ? L : T;
    dim3 grid(cdiv(T, 128), rows, nslab);
    k_mw_extend<<<grid, 128, 0, st>>>(L, slab_n, mwss, pair, ldin, ldout, Fa, Fa_slab, X, X_slab);
    count_bytes(16.0 * (double)T * ((double)T + rows) * nslab); LAUNCHED(); return cudaSuccess;
}
cudaError_t st_mw_pad_phase(int L, int nslab, int mwss, int rows, int ldin, int ldout, const double2* Y, size_t Y_slab, double2* Z, size_t Z_slab,
                            cudaStream_t st) {
    const int T = mwss ? 2 * L : 2 * L - 1;
    dim3 grid(cdiv(ldout, 128), rows, nslab);
    k_mw_pad_phase<<<grid, 128, 0, st>>>(L, mwss, ldin, ldout, Y, Y_slab, Z, Z_slab);
    count_bytes(16.0 * (double)rows * ((double)T + ldout) * nslab); LAUNCHED(); return cudaSuccess;
}
cudaError_t st_weight_split(int L, int NBin, int ldin, int pair, int nth, int ntp, int NC, int mmin, int npass, const double* wq, const double2* U,
                            size_t U_slab, const ThetaPass* passes, int th_lo, int th_hi, cudaStream_t st) {
    if (npass == 0) return cudaSuccess;
    dim3 grid(cdiv(ntp, 128), L - mmin - 1, npass);
    k_weight_split<<<grid, 128, 0, st>>>(L, NBin, ldin, pair, nth, ntp, NC, wq, U, U_slab, passes, th_lo, th_hi);
    count_bytes(32.0 * NC * (double)(L - mmin - 1) * ntp * npass); LAUNCHED(); return cudaSuccess;
}
cudaError_t st_pole_forward(int L, int Lp, int n, int north, int NBin, int ldin, int col, double w, const double2* U, double2* H,
                            cudaStream_t st) {
    k_pole_forward<<<cdiv(L, 128), 128, 0, st>>>(L, Lp, n, north, NBin, ldin, col, w, U, H);
    count_bytes(32.0 * L); LAUNCHED(); return cudaSuccess;
}
cudaError_t st_finalize_forward(int L, int Lp, int nslab, const int* slab_n, const int* cslab, int real, const double* scale, const double2* H,
                                size_t H_slab, double2* coef, size_t coef_slab, cudaStream_t st) {
    dim3 grid(cdiv(2 * L - 1, 32), cdiv(L, 32), nslab), block(32, 8);
    k_finalize_forward<<<grid, block, 0, st>>>(L, Lp, slab_n, cslab, real, scale, H, H_slab, coef, coef_slab);
    count_bytes(32.0 * (double)(2 * L - 1) * L * nslab); LAUNCHED(); return cudaSuccess;
}
cudaError_t st_rows_reorder(int L, int NB, int ncol, int ldsrc, int lddst, int to_mi, const double2* src, double2* dst, cudaStream_t st) {
    dim3 grid(cdiv(ncol, 128), 2 * L - 1);      // rows r = m + L - 1 of the m-ordered array; NB = number of phi bins of the other one
    k_rows_bin_to_mi<<<grid, 128, 0, st>>>(L, NB, ncol, ldsrc, lddst, to_mi, src, dst);
    count_bytes(32.0 * (double)(2 * L - 1) * ncol); LAUNCHED(); return cudaSuccess;
}
cudaError_t st_transpose_slabs(int nslab, int nrow, int ncol, int ldin, int ldout, const double2* in, size_t in_slab, double2* out,
                               size_t out_slab, cudaStream_t st) {
    k_transpose_slabs<<<dim3(cdiv(ncol, 32), cdiv(nrow, 32), nslab), dim3(32, 8), 0, st>>>(nrow, ncol, ldin, ldout, in, in_slab, out, out_slab);
    count_bytes(32.0 * (double)nrow * ncol * nslab); LAUNCHED(); return cudaSuccess;
}
cudaError_t st_scale_copy(size_t n, double s, const double2* in, double2* out, cudaStream_t st) {
    k_scale_copy<<<cdiv(n, 256), 256, 0, st>>>(n, s, in, out);
    count_bytes(32.0 * (double)n); LAUNCHED(); return cudaSuccess;
}
cudaError_t st_prep_inverse_batch(int L, int Lp, int NC, int B, int ncg, int n, int sgn_out, int m_end, int mmin, const double2* coef,
                                  const double* scale, const double* C, const double2* SG, int sgstride, double* Gb, size_t cg_stride,
                                  cudaStream_t st) {
    dim3 grid(cdiv(Lp, 16), cdiv(L - m_end, 8), ncg);
    k_prep_inverse_batch<<<grid, 128, 0, st>>>(L, Lp, NC, B, n, sgn_out, m_end, mmin, coef, scale, C, SG, sgstride, Gb, cg_stride);
    count_bytes(16.0 * B * NC * (double)(L - m_end) * L + 8.0 * SHT_MMA_ROW * (double)ncg * (L - m_end) * Lp); LAUNCHED(); return cudaSuccess;
}
cudaError_t st_weight_split_batch(int L, int NBin, int ldin, int pair, size_t U_slab, int nth, int ntp, int NC, int B, int ncg, int n, int sgn_out,
                                  int m_end, int fold, const int* m_lo, const double* wq, const double* lam, const double2* U, double* Wb,
                                  size_t cg_stride, cudaStream_t st) {
    dim3 grid(cdiv(ntp, 32), L - m_end, ncg);
    k_weight_split_batch<<<grid, 128, 0, st>>>(L, NBin, ldin, pair, U_slab, nth, ntp, NC, B, n, sgn_out, m_end, fold, m_lo, wq, lam, U, Wb, cg_stride);
    count_bytes(16.0 * B * NC * (double)(L - m_end) * ntp + 8.0 * SHT_MMA_ROW * (double)ncg * (L - m_end) * ntp); LAUNCHED(); return cudaSuccess;
}
cudaError_t st_unpack_batch(int L, int Lp, int Mp, int mlim, int NC, int B, int ncg, int n, int sgn_out, int m_end, int mmin, int fwd, int fold,
                            const double* C, const double* Ob, size_t cg_stride, double2* out, size_t out_slab, int ld, cudaStream_t st) {
    dim3 grid(cdiv(Mp, 32), L - m_end, ncg);
    k_unpack_batch<<<grid, 128, 0, st>>>(L, Lp, Mp, mlim, NC, B, n, sgn_out, m_end, mmin, fwd, fold, C, Ob, cg_stride, out, out_slab, ld);
    count_bytes(8.0 * SHT_MMA_NCOL * (double)ncg * (L - m_end) * Mp + 32.0 * B * NC * (double)(L - m_end) * mlim); LAUNCHED(); return cudaSuccess;
}
cudaError_t st_weight_split_fold0(int L, int NBin, int ldin, int pair, int nth, int ntp, int nfull, int NC, int m_end, const double* wq,
                                  const double2* U, double2* W, int th_lo, int th_hi, cudaStream_t st) {
    dim3 grid(cdiv(ntp, 128), L - m_end);
    k_weight_split_fold0<<<grid, 128, 0, st>>>(L, NBin, ldin, pair, nth, ntp, nfull, NC, m_end, wq, U, W, th_lo, th_hi);
    count_bytes(64.0 * NC * (double)(L - m_end) * ntp); LAUNCHED(); return cudaSuccess;
}
cudaError_t st_weight_split_batch_fold0(int L, int NBin, int ldin, int pair, size_t U_slab, int nth, int ntp, int nfull, int NC, int B, int ncg,
                                        int m_end, const double* wq, const double* lam, const double2* U, double* Wb, size_t cg_stride,
                                        cudaStream_t st) {
    dim3 grid(cdiv(ntp, 32), L - m_end, ncg);
    k_weight_split_batch_fold0<<<grid, 128, 0, st>>>(L, NBin, ldin, pair, U_slab, nth, ntp, nfull, NC, B, m_end, wq, lam, U, Wb, cg_stride);
    count_bytes(32.0 * B * NC * (double)(L - m_end) * ntp + 8.0 * SHT_MMA_ROWF * (double)ncg * (L - m_end) * ntp); LAUNCHED(); return cudaSuccess;
}
cudaError_t st_ab32(int L, int Lp, float4* AB, cudaStream_t st) {
    k_ab32<<<dim3(cdiv(Lp, 128), L), 128, 0, st>>>(L, Lp, AB);
    LAUNCHED(); return cudaSuccess;
}
cudaError_t st_start32(size_t n, const double* v64, const uint8_t* k64, float* v32, uint16_t* k16, cudaStream_t st) {
    k_start32<<<cdiv(n, 256), 256, 0, st>>>(n, v64, k64, v32, k16);
    LAUNCHED(); return cudaSuccess;
}
cudaError_t st_prep_inverse_f32(int L, int Lp, int NC, const double2* coef, const double* scale, float2* G, cudaStream_t st) {
    dim3 grid(cdiv(Lp, 32), cdiv(L, 32)), block(32, 8);
    k_prep_inverse_f32<<<grid, block, 0, st>>>(L, Lp, NC, coef, scale, reinterpret_cast<float4*>(G));
    count_bytes(16.0 * NC * (double)L * L + 16.0 * NC * (double)L * Lp); LAUNCHED(); return cudaSuccess;
}
cudaError_t st_weight_split_f32(int L, int NBin, int ldin, int pair, int nth, int ntp, int NC, const double* wq, const double2* U, float2* W,
                                cudaStream_t st) {
    k_weight_split_f32<<<dim3(cdiv(ntp, 128), L), 128, 0, st>>>(L, NBin, ldin, pair, nth, ntp, NC, wq, U, reinterpret_cast<float*>(W));
    count_bytes(24.0 * NC * (double)L * ntp); LAUNCHED(); return cudaSuccess;
}
cudaError_t st_f32_to_f64(size_t n, const float* in, double* out, cudaStream_t st) {
    k_c64_to_c128<<<cdiv(n, 256), 256, 0, st>>>(n, in, out);
    count_bytes(12.0 * (double)n); LAUNCHED(); return cudaSuccess;
}
cudaError_t st_f64_to_f32(size_t n, const double* in, float* out, cudaStream_t st) {
    k_c128_to_c64<<<cdiv(n, 256), 256, 0, st>>>(n, in, out);
    count_bytes(12.0 * (double)n); LAUNCHED(); return cudaSuccess;
}
cudaError_t st_weight_split_f32_fold0(int L, int NBin, int ldin, int pair, int nth, int ntp, int nfull, int NC, const double* wq, const double2* U,
                                      float2* W, cudaStream_t st) {
    k_weight_split_f32_fold0<<<dim3(cdiv(ntp, 128), L), 128, 0, st>>>(L, NBin, ldin, pair, nth, ntp, nfull, NC, wq, U, reinterpret_cast<float*>(W));
    count_bytes(48.0 * NC * (double)L * ntp); LAUNCHED(); return cudaSuccess;
}
cudaError_t st_sym_extend(int L, int n, int pair, int ldin, const double2* F, double2* X, cudaStream_t st) {
    const int rows = pair ? L : 2 * L - 1;
    k_sym_extend<<<dim3(cdiv(2 * L, 128), rows), 128, 0, st>>>(L, n, pair, ldin, F, X);
    count_bytes(16.0 * (double)(2 * L) * ((double)rows + 0.5 * (2 * L - 1))); LAUNCHED(); return cudaSuccess;
}
cudaError_t st_sym_rebin(int L, int rows, const double2* Y, double2* Z, cudaStream_t st) {
    k_sym_rebin<<<dim3(cdiv(2 * L - 1, 128), rows), 128, 0, st>>>(L, Y, Z);
    count_bytes(32.0 * (double)(2 * L - 1) * rows); LAUNCHED(); return cudaSuccess;
}
cudaError_t st_sym_unpair(int L, int n, int ldout, const double2* X, double2* F, cudaStream_t st) {
    k_sym_unpair<<<dim3(cdiv(L, 128), 2 * L - 1), 128, 0, st>>>(L, n, ldout, X, F);
    count_bytes(16.0 * (double)(2 * L - 1) * (2.0 * L)); LAUNCHED(); return cudaSuccess;
}
cudaError_t st_rows_head(int nrows, int ncol, int ldin, int ldout, const double2* in, double2* out, cudaStream_t st) {
    k_rows_head<<<dim3(cdiv(ncol, 128), nrows), 128, 0, st>>>(ncol, ldin, ldout, in, out);
    count_bytes(32.0 * (double)nrows * ncol); LAUNCHED(); return cudaSuccess;
}
cudaError_t st_scale_rows(int nrow, int ncol, double sgn, const double* d, const double2* in, double2* out, cudaStream_t st) {
    k_scale_rows<<<dim3(cdiv(ncol, 128), nrow), 128, 0, st>>>(nrow, ncol, sgn, d, in, out);
    count_bytes(32.0 * (double)nrow * ncol); LAUNCHED(); return cudaSuccess;
}
cudaError_t st_scale_cols(int nrows, int ncol, int ld, const double* w, double2* F, cudaStream_t st) {
    k_scale_cols<<<dim3(cdiv(ncol, 128), nrows), 128, 0, st>>>(ncol, ld, w, F);
    count_bytes(32.0 * (double)nrows * ncol); LAUNCHED(); return cudaSuccess;
}
cudaError_t st_adj_weight_pad(int L, int NBq, int ldq, const double2* Fq, const double* wq, int NB, int T2, double2* Z, cudaStream_t st) {
    k_adj_weight_pad<<<dim3(cdiv(T2, 128), NB), 128, 0, st>>>(L, NBq, ldq, Fq, wq, NB, T2, Z);
    count_bytes(16.0 * (double)NB * (2.0 * L + T2)); LAUNCHED(); return cudaSuccess;
}
cudaError_t st_adj_trunc_phase(int L, int mwss, int NB, int T2, const double2* Zf, double2* X, cudaStream_t st) {
    const int T = mwss ? 2 * L : 2 * L - 1;
    k_adj_trunc_phase<<<dim3(cdiv(T, 128), NB), 128, 0, st>>>(L, mwss, T2, Zf, X);
    count_bytes(32.0 * (double)NB * T); LAUNCHED(); return cudaSuccess;
}
cudaError_t st_adj_fold(int L, int n, int mwss, int NB, int nrmap, int ldf, const double2* X, double2* F, cudaStream_t st) {
    k_adj_fold<<<dim3(cdiv(nrmap, 128), NB), 128, 0, st>>>(L, n, mwss, nrmap, ldf, X, F);
    count_bytes(16.0 * (double)NB * (3.0 * nrmap)); LAUNCHED(); return cudaSuccess;
}
cudaError_t st_vec_sub(size_t n, const double* a, const double* b, double* out, cudaStream_t st) {
    k_vec_sub<<<cdiv(n, 256), 256, 0, st>>>(n, a, b, out);
    count_bytes(24.0 * (double)n); LAUNCHED(); return cudaSuccess;
}
cudaError_t st_vec_add(size_t n, const double* x, double* y, cudaStream_t st) {
    k_vec_add<<<cdiv(n, 256), 256, 0, st>>>(n, x, y);
    count_bytes(24.0 * (double)n); LAUNCHED(); return cudaSuccess;
}
