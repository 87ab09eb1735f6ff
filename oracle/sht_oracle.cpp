// sht_oracle.cpp -- CPU ORACLE for the spin spherical harmonic / Wigner transforms of arXiv 2311.14670.
//
// THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and bench.py's
// cpu_baseline / --impl reference legs may build, load or call it.  It shares no code, header, table or
// constant generator with the CUDA path under paper_2311_14670_b200/csrc and neither side includes the other.
//
// What it computes: the *plain definitions* of the four maps of PAPER.md:168 (Sec. 2.4),
//   inverse  f(theta,phi)   = sum_{l,m} flm  sY_lm(theta,phi)                       (Eq. 4 truncated at L)
//   forward  flm            ~ sum_{theta,phi} q f conj(sY_lm)                       (Eq. 19)
//   inverse  f(a,b,g)       = sum_l (2l+1)/(8pi^2) sum_{m,n} flmn conj(D^l_mn)      (Eq. 13)
//   forward  flmn           ~ sum q f D^l_mn                                        (Eq. 20)
// with  sY_lm = (-1)^s sqrt((2l+1)/4pi) d^l_{m,-s}(theta) e^{i m phi}  (Eq. 9+10) and
// D^l_mn = e^{-i m alpha} d^l_mn(beta) e^{-i n gamma} (Eq. 10).  Sums are evaluated by direct summation in
// `long double`, in the separated order of Eq. 30-33 (an exact re-association; the un-separated O(L^4) sums are
// also provided for tiny L and compared in the tests).  All DFTs are naive O(n^2) sums with exactly reduced angles.
//
// The Wigner d-functions are obtained by routes that NEVER recurse in m (the paper's method, Eq. 25, does):
//   E  explicit Wigner sum (equivalent to Eq. 21/22)             -- tiny l only
//   R  Risbo's half-integer-step recursion (ref. [57] of the paper)   -- any beta, O(L^3) per beta
//   T  three-term recurrence in l at fixed (m,n) with explicit exponent tracking    -- the route the transforms use
// E, R and T are cross-checked against each other and against closed forms in tests/test_oracle_wigner.py.
//
// MW forward transform: PAPER.md:379-381 (Sec. 4.2.2) -- extend F_m(theta) to the torus with sign (-1)^{m+s},
// upsample by zero padding in theta-Fourier space to the MW grid of band-limit 2L, integrate with the weights of
// Eq. 41-44 taken at band-limit 2L (closed form, reading R9).  HEALPix: PAPER.md:399-407 (weights
// 4pi/Npix; ring geometry from the public definition of the scheme, reading R11).
//
// Further samplings: DH Eq. 34-36, MWSS Eq. 39-40 with the unified weights Eq. 43-44
// (PAPER.md:349-381), Gauss-Legendre Eq. 45-46 (Eq. 46 as printed is not the Gauss-Legendre weight -- reading
// R22 of DESIGN.md: the standard weight 2/((1-x^2) P_L'(x)^2) is used and pinned against numpy's leggauss).
// Adjoints (Eq. 52 / 58): the plain conjugate-transposed sums of the forward / inverse
// transforms above, step by step in reverse order (orc_s2_forward_adjoint, orc_s2_inverse_adjoint_columns); pinned by the
// dot-product identity <F x, y> = <x, F^H y> against the pinned transforms and by Eq. 52 / 58 on the direct-quadrature samplings.
//
// Parity pins (tests, -m "not gpu"): closed-form Y_lm / sY_lm, scipy sph_harm_y, Jacobi form (Eq. 22) through
// scipy/mpmath, d(0)=I, d(pi), symmetries, orthogonality, E==R==T, un-separated sums, quadrature exactness,
// exact MW / SO(3) round trips (sampling theorem).  HEALPix forward: the scheme has no sampling theorem, so it is
// pinned by normalisation (constant map), geometry, the shared, pinned, Y_lm, and by CONVERGENCE: the forward of a synthesised
// band-limited map converges to the generating coefficients at second order in the pixel size (error / 4 per doubling of nside),
// test_oracle_s2.py::test_healpix_forward_converges_to_the_generating_coefficients; see DESIGN.md.
//
// Build: python oracle/build.py   (g++ -O2 -fopenmp -shared -fPIC)
#include <cmath>
#include <cstdint>
#include <cstdlib>
#include <cstring>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef long double ld;
static const ld PI_L = 3.14159265358979323846264338327950288419716939937510L;

struct cld { ld re, im; };
static inline cld cmul(cld a, cld b) { return {a.re * b.re - a.im * b.im, a.re * b.im + a.im * b.re}; }
static inline cld cadd(cld a, cld b) { return {a.re + b.re, a.im + b.im}; }
static inline cld cscale(cld a, ld s) { return {a.re * s, a.im * s}; }
static inline ld sgn_pow(long k) { return (k & 1L) ? -1.0L : 1.0L; }  // (-1)^k, k may be negative

// e^{2 pi i k / n} with the angle reduced exactly (k mod n) before any floating point is touched.
static inline cld unit_root(long k, long n) {
    long r = k % n; if (r < 0) r += n;
    ld a = 2.0L * PI_L * (ld)r / (ld)n;
    return {cosl(a), sinl(a)};
}
// e^{i pi k / n}, angle reduced mod 2n.
static inline cld unit_root_pi(long k, long n) {
    long r = k % (2 * n); if (r < 0) r += 2 * n;
    ld a = PI_L * (ld)r / (ld)n;
    return {cosl(a), sinl(a)};
}

// ------------------------------------------------------------------------------------------------------------
// Sampling: iso-latitude rings.  Half-angle trigonometry is carried explicitly so that nothing
// is lost near the poles.
// ------------------------------------------------------------------------------------------------------------
struct Ring {
    ld ct, st;      // cos(theta), sin(theta)
    ld c2, s2;      // cos(theta/2), sin(theta/2)
    int nphi;       // samples on the ring
    ld phi0;        // first sample longitude; phi_p = phi0 + 2 pi p / nphi
    ld w;           // quadrature weight q(theta,phi) of one sample of this ring (0 if the ring set carries none)
    int pole;       // 0 regular, 1 theta = 0, 2 theta = pi  (Eq. 28/29 are used there)
    long off;       // offset of the ring's first sample in the ring-ordered map
};
struct RingSet { std::vector<Ring> r; long npix; };

// MW sample positions, Eq. 37-38: theta_t = (2t+1)pi/(2L-1), t<L; phi_p = 2 pi p/(2L-1).
// `nphi` is passed separately because the quadrature grid (band-limit 2L in theta) keeps the 2L-1 longitudes.
static RingSet rings_mw(int Lt, int nphi) {
    RingSet S; S.r.resize(Lt); long off = 0;
    for (int t = 0; t < Lt; ++t) {
        Ring& g = S.r[t];
        ld th = PI_L * (ld)(2 * t + 1) / (ld)(2 * Lt - 1);
        g.pole = (t == Lt - 1) ? 2 : 0;
        g.ct = cosl(th); g.st = sinl(th); g.c2 = cosl(th / 2); g.s2 = sinl(th / 2);
        if (g.pole == 2) { g.ct = -1; g.st = 0; g.c2 = 0; g.s2 = 1; }
        g.nphi = nphi; g.phi0 = 0; g.w = 0; g.off = off; off += nphi;
    }
    S.npix = off; return S;
}
// theta-quadrature weights v_u for integrating (even, torus-band-limit 2Lq-1) integrands against sin(theta) on
// the MW grid of band-limit Lq: Eq. 41-44 with reflection sign +1 (R9):
//   v_u = (1/(2Lq-1)) * zeta_u * sum_{j : |2j| <= Lq-1} [2/(1-4j^2)] * 2cos(2 j theta_u),  zeta = 1 (regular), 1/2 (pole)
static void mw_theta_weights(int Lq, std::vector<ld>& v) {
    v.assign(Lq, 0);
    int T = 2 * Lq - 1, jmax = (Lq - 1) / 2;
    for (int u = 0; u < Lq; ++u) {
        ld acc = 0;
        for (int j = -jmax; j <= jmax; ++j) {
            // cos(2 j theta_u) = Re e^{i pi 2j(2u+1)/T}
            cld e = unit_root_pi((long)2 * j * (2 * u + 1), T);
            acc += (2.0L / (1.0L - 4.0L * (ld)j * (ld)j)) * 2.0L * e.re;
        }
        v[u] = acc / (ld)T;
        if (u == Lq - 1) v[u] *= 0.5L;
    }
}
// HEALPix ring scheme (Gorski et al., ref. [43]).  Rings r = 1..4 nside-1 north to south.
static RingSet rings_healpix(int nside) {
    RingSet S; int nr = 4 * nside - 1; S.r.resize(nr); long off = 0;
    ld ns = (ld)nside; ld npix = 12.0L * ns * ns;
    for (int i = 0; i < nr; ++i) {
        int r = i + 1; Ring& g = S.r[i]; ld z; int rr = r;
        bool south = r > 2 * nside;
        if (south) rr = 4 * nside - r;            // mirror ring
        if (rr < nside) { z = 1.0L - (ld)rr * (ld)rr / (3.0L * ns * ns); g.nphi = 4 * rr; g.phi0 = PI_L / (ld)g.nphi; }
        else { z = 4.0L / 3.0L - 2.0L * (ld)rr / (3.0L * ns); g.nphi = 4 * nside; g.phi0 = ((rr - nside) % 2 == 0) ? PI_L / (ld)g.nphi : 0.0L; }
        if (r == 2 * nside) z = 0;
        if (south) z = -z;
        g.ct = z; g.st = sqrtl((1 - z) * (1 + z));
        g.s2 = sqrtl((1 - z) / 2); g.c2 = sqrtl((1 + z) / 2);
        g.pole = 0; g.w = 4.0L * PI_L / npix; g.off = off; off += g.nphi;
    }
    S.npix = off; return S;
}

// DH sample positions and weights, Eq. 34-36: theta_t = (2t+1)pi/(4L), t < 2L; phi_p = 2 pi p/(2L-1);
//   q(theta) = (4 pi/(L(2L-1))) sin(theta) sum_{k=0}^{L-1} sin((2k+1)theta)/(2k+1).
static RingSet rings_dh(int L) {
    RingSet S; S.r.resize(2 * L); long off = 0;
    for (int t = 0; t < 2 * L; ++t) {
        Ring& g = S.r[t];
        ld th = PI_L * (ld)(2 * t + 1) / (ld)(4 * L);
        g.pole = 0; g.ct = cosl(th); g.st = sinl(th); g.c2 = cosl(th / 2); g.s2 = sinl(th / 2);
        ld acc = 0;
        for (int k = L - 1; k >= 0; --k) {
            // sin((2k+1) theta_t) = Im e^{i pi (2k+1)(2t+1)/(4L)}, angle reduced exactly
            acc += unit_root_pi((long)(2 * k + 1) * (2 * t + 1), 4 * L).im / (ld)(2 * k + 1);
        }
        g.w = 4.0L * PI_L / ((ld)L * (ld)(2 * L - 1)) * g.st * acc;
        g.nphi = 2 * L - 1; g.phi0 = 0; g.off = off; off += g.nphi;
    }
    S.npix = off; return S;
}
// MWSS sample positions, Eq. 39-40: theta_t = 2 pi t/(2Lt), t = 0..Lt (both poles are rings);
// phi_p = 2 pi p/nphi.  `nphi` is passed separately: the quadrature grid of band-limit 2L keeps the 2L longitudes.
static RingSet rings_mwss(int Lt, int nphi) {
    RingSet S; S.r.resize(Lt + 1); long off = 0;
    for (int t = 0; t <= Lt; ++t) {
        Ring& g = S.r[t];
        ld th = PI_L * (ld)t / (ld)Lt;
        g.pole = (t == 0) ? 1 : (t == Lt) ? 2 : 0;
        g.ct = cosl(th); g.st = sinl(th); g.c2 = cosl(th / 2); g.s2 = sinl(th / 2);
        if (g.pole == 1) { g.ct = 1; g.st = 0; g.c2 = 1; g.s2 = 0; }
        if (g.pole == 2) { g.ct = -1; g.st = 0; g.c2 = 0; g.s2 = 1; }
        if (2 * t == Lt) { g.ct = 0; g.st = 1; }                      // the equator ring of an even Lt, exactly
        g.nphi = nphi; g.phi0 = 0; g.w = 0; g.off = off; off += nphi;
    }
    S.npix = off; return S;
}
// MWSS theta-quadrature weights at band-limit Lq (T = 2Lq samples on the theta circle), Eq. 41-44 with reflection sign +1
// (R9: the integrand of the transform is even under theta -> 2pi - theta, so the odd terms w^(+-1) cancel):
//   v_u = (1/T) (1 + zeta_u) sum_{j : |2j| <= Lq-1} [2/(1-4j^2)] cos(2 j theta_u),   zeta_u = 0 at the poles u = 0, Lq, else 1.
static void mwss_theta_weights(int Lq, std::vector<ld>& v) {
    v.assign(Lq + 1, 0);
    int T = 2 * Lq, jmax = (Lq - 1) / 2;
    for (int u = 0; u <= Lq; ++u) {
        ld acc = 0;
        for (int j = -jmax; j <= jmax; ++j) acc += (2.0L / (1.0L - 4.0L * (ld)j * (ld)j)) * unit_root((long)2 * j * u, T).re;
        v[u] = acc / (ld)T * ((u == 0 || u == Lq) ? 1.0L : 2.0L);
    }
}
// Gauss-Legendre rings: theta_t = acos(x_t), x_t the roots of P_L, north to south; phi_p = 2 pi p/(2L-1), Eq. 45.
// Roots by Newton's iteration in theta on P_L(cos theta) (three-term recurrence), so that half-angle trigonometry keeps full
// relative accuracy near the poles.  Weights: 2/((1-x^2) P_L'(x)^2) times q_Phi = 2 pi/(2L-1)  (reading R22 of Eq. 46).
static void legendre_pl(int L, ld x, ld& p, ld& dp) {      // P_L(x) and P_L'(x)
    ld p0 = 1, p1 = x;
    if (L == 0) { p = 1; dp = 0; return; }
    for (int k = 2; k <= L; ++k) { ld pk = ((ld)(2 * k - 1) * x * p1 - (ld)(k - 1) * p0) / (ld)k; p0 = p1; p1 = pk; }
    p = p1; dp = (ld)L * (x * p1 - p0) / (x * x - 1);
}
static RingSet rings_gl(int L) {
    RingSet S; S.r.resize(L); long off = 0;
    for (int t = 0; t < L; ++t) {
        Ring& g = S.r[t];
        ld th = PI_L * ((ld)t + 0.75L) / ((ld)L + 0.5L);              // Tricomi-type initial guess for the (t+1)-th root
        ld p, dp;
        for (int it = 0; it < 100; ++it) {
            legendre_pl(L, cosl(th), p, dp);
            ld dth = p / (sinl(th) * dp);                               // d/dtheta P_L(cos theta) = -sin(theta) P_L'
            th += dth;
            if (fabsl(dth) < 1e-19L * th) break;
        }
        if (2 * t + 1 == L) th = PI_L / 2;                              // the equator root of an odd L, exactly
        legendre_pl(L, cosl(th), p, dp);
        g.pole = 0; g.ct = cosl(th); g.st = sinl(th); g.c2 = cosl(th / 2); g.s2 = sinl(th / 2);
        if (2 * t + 1 == L) { g.ct = 0; g.st = 1; }
        g.w = 2.0L * PI_L / (ld)(2 * L - 1) * 2.0L / (g.st * g.st * dp * dp);
        g.nphi = 2 * L - 1; g.phi0 = 0; g.off = off; off += g.nphi;
    }
    S.npix = off; return S;
}

// ------------------------------------------------------------------------------------------------------------
// Provider E: Wigner's explicit sum (Varshalovich convention, first index m; d^1_{10} = -sin(beta)/sqrt 2).
//   d^l_mn = sqrt((l+n)!(l-n)!(l+m)!(l-m)!) sum_k (-1)^{k-n+m} cos^{2l-2k+n-m}(b/2) sin^{2k-n+m}(b/2)
//                                               / ((l+n-k)! k! (l-k-m)! (k-n+m)!)
// ------------------------------------------------------------------------------------------------------------
static ld fact(int k) { ld f = 1; for (int i = 2; i <= k; ++i) f *= (ld)i; return f; }
static ld d_explicit_hs(int l, int m, int n, ld c, ld s) {
    if (abs(m) > l || abs(n) > l) return 0;
    int k0 = (n - m > 0) ? n - m : 0, k1 = (l + n < l - m) ? l + n : l - m;
    ld pre = sqrtl(fact(l + n) * fact(l - n) * fact(l + m) * fact(l - m)), sum = 0;
    for (int k = k0; k <= k1; ++k) {
        ld t = sgn_pow(k - n + m) / (fact(l + n - k) * fact(k) * fact(l - k - m) * fact(k - n + m));
        int pc = 2 * l - 2 * k + n - m, ps = 2 * k - n + m;
        ld cp = 1, sp = 1;
        for (int i = 0; i < pc; ++i) cp *= c;
        for (int i = 0; i < ps; ++i) sp *= s;
        sum += t * cp * sp;
    }
    return pre * sum;
}
// (long double scalars cross the C ABI by pointer: ctypes would round by-value long doubles to double)
extern "C" void orc_d_explicit(int l, int m, int n, const long double* beta, long double* out) {
    *out = d_explicit_hs(l, m, n, cosl(*beta / 2), sinl(*beta / 2));
}

// ------------------------------------------------------------------------------------------------------------
// Provider R: Risbo's recursion (J = 2j runs over half-integer steps).  Plane J is (J+1)x(J+1), index
// [i][k] = (m + j, n + j).  Integer planes (J even) are copied out: out[l][(m+l)*(2l+1) + (n+l)], packed per l
// at offset sum_{l'<l} (2l'+1)^2.
//   J d^J[i][k] = sqrt((J-i)(J-k)) c P[i][k] - sqrt(i (J-k)) s P[i-1][k] + sqrt((J-i) k) s P[i][k-1] + sqrt(i k) c P[i-1][k-1]
// ------------------------------------------------------------------------------------------------------------
extern "C" void orc_d_risbo(int L, const long double* beta_p, long double* out) {
    ld beta = *beta_p;
    ld c = cosl(beta / 2), s = sinl(beta / 2);
    std::vector<ld> P(1, 1.0L), Q;
    long off = 0;
    out[off] = 1; off += 1;                       // l = 0
    for (int J = 1; J <= 2 * (L - 1); ++J) {
        int n1 = J + 1, n0 = J;                   // new / previous plane sizes
        Q.assign((size_t)n1 * n1, 0);
        for (int i = 0; i <= J; ++i) for (int k = 0; k <= J; ++k) {
            ld v = 0;
            if (i < n0 && k < n0)   v += sqrtl((ld)(J - i) * (ld)(J - k)) * c * P[(size_t)i * n0 + k];
            if (i >= 1 && k < n0)   v -= sqrtl((ld)i * (ld)(J - k)) * s * P[(size_t)(i - 1) * n0 + k];
            if (i < n0 && k >= 1)   v += sqrtl((ld)(J - i) * (ld)k) * s * P[(size_t)i * n0 + (k - 1)];
            if (i >= 1 && k >= 1)   v += sqrtl((ld)i * (ld)k) * c * P[(size_t)(i - 1) * n0 + (k - 1)];
            Q[(size_t)i * n1 + k] = v / (ld)J;
        }
        P.swap(Q);
        if (J % 2 == 0) { memcpy(out + off, P.data(), sizeof(ld) * (size_t)n1 * n1); off += (long)n1 * n1; }
    }
}

// ------------------------------------------------------------------------------------------------------------
// Provider T: recurrence in l at fixed (m,n):
//   d^{l+1}_mn = [ (2l+1)(l(l+1) cos b - m n) d^l_mn - (l+1) sqrt((l^2-m^2)(l^2-n^2)) d^{l-1}_mn ]
//                / [ l sqrt(((l+1)^2-m^2)((l+1)^2-n^2)) ],      d^1_00 = cos b for the l = 0 step,
// started at l0 = max(|m|,|n|) from the closed form Eq. 27 moved to the right corner with the
// symmetries d_mn = (-1)^{m-n} d_nm = (-1)^{m-n} d_{-m,-n} = d_{-n,-m}, with d^{l0-1} = 0.
// The start value can be as small as 1e-35000, so the pair is carried as value * 2^e with an explicit int e.
// l(l+1)cos b - mn is formed without cancellation from the half angle: (l(l+1)-mn) - 2l(l+1)s2^2 on the northern
// hemisphere, -(l(l+1)+mn) + 2l(l+1)c2^2 on the southern.
// out[l] for l in [0,L): true value (0 where it underflows long double or l < l0).
// ------------------------------------------------------------------------------------------------------------
// log2 of Eq. 27's magnitude: d^l_{l,k} = sqrt((2l)!/((l+k)!(l-k)!)) (-s2)^{l-k} c2^{l+k}
static void top_value(int l, int k, ld c2, ld s2, ld& mant, long& e2) {
    // binomial (2l choose l-k) as an exact running product with exponent tracking (no lgamma: DESIGN.md R7)
    ld p = 1; long e = 0; int ex;
    for (int i = 1; i <= l - k; ++i) {
        p *= (ld)(l + k + i) / (ld)i;
        p = frexpl(p, &ex); e += ex;
    }
    // sqrt: make exponent even
    if (e & 1L) { p *= 2; e -= 1; }
    p = sqrtl(p); e /= 2;
    ld base[2] = {s2, c2}; int pw[2] = {l - k, l + k};
    for (int b = 0; b < 2; ++b) {
        // x^n by repeated squaring with exponent tracking
        ld x = frexpl(base[b], &ex); long xe = ex; int nn = pw[b];
        ld r = 1; long re = 0;
        while (nn > 0) {
            if (nn & 1) { r *= x; re += xe; r = frexpl(r, &ex); re += ex; }
            x *= x; xe *= 2; x = frexpl(x, &ex); xe += ex; nn >>= 1;
        }
        p *= r; e += re; p = frexpl(p, &ex); e += ex;
    }
    mant = p * sgn_pow(l - k); e2 = e;
}
static void d_lrec(int L, int m, int n, const Ring& g, ld* out) {
    for (int l = 0; l < L; ++l) out[l] = 0;
    int am = abs(m), an = abs(n), l0 = am > an ? am : an;
    if (l0 >= L) return;
    if (g.pole == 1) { if (m == n) for (int l = l0; l < L; ++l) out[l] = 1; return; }                       // Eq. 28
    if (g.pole == 2) { if (m == -n) for (int l = l0; l < L; ++l) out[l] = sgn_pow(l + m); return; }         // Eq. 29
    ld cur; long e;
    if (m == l0)        { top_value(l0, n, g.c2, g.s2, cur, e); }
    else if (m == -l0)  { top_value(l0, -n, g.c2, g.s2, cur, e); cur *= sgn_pow(-l0 - n); }
    else if (n == l0)   { top_value(l0, m, g.c2, g.s2, cur, e); cur *= sgn_pow(m - l0); }
    else                { top_value(l0, -m, g.c2, g.s2, cur, e); }
    ld prev = 0;
    const long EMIN = -16300;
    bool north = g.ct >= 0;
    ld mn = (ld)m * (ld)n;
    for (int l = l0;; ++l) {
        out[l] = (e < EMIN) ? 0.0L : ldexpl(cur, (int)e);
        if (l + 1 >= L) break;
        ld nxt;
        if (l == 0) nxt = g.ct * cur;
        else {
            ld ll1 = (ld)l * (ld)(l + 1);
            ld x = north ? (ll1 - mn) - 2 * ll1 * g.s2 * g.s2 : -(ll1 + mn) + 2 * ll1 * g.c2 * g.c2;
            ld l2 = (ld)l * (ld)l, lp2 = (ld)(l + 1) * (ld)(l + 1), m2 = (ld)m * (ld)m, n2 = (ld)n * (ld)n;
            ld num = (ld)(2 * l + 1) * x * cur - (ld)(l + 1) * sqrtl((l2 - m2) * (l2 - n2)) * prev;
            nxt = num / ((ld)l * sqrtl((lp2 - m2) * (lp2 - n2)));
        }
        prev = cur; cur = nxt;
        if (fabsl(cur) > 0x1p+2000L) { cur *= 0x1p-2000L; prev *= 0x1p-2000L; e += 2000; }
    }
}
extern "C" void orc_d_lrec(int L, int m, int n, const long double* half /*{cos(b/2), sin(b/2)}*/, long double* out) {
    ld cos_half = half[0], sin_half = half[1];
    Ring g; g.c2 = cos_half; g.s2 = sin_half; g.ct = (cos_half - sin_half) * (cos_half + sin_half);
    g.st = 2 * cos_half * sin_half; g.pole = 0; g.nphi = 0; g.phi0 = 0; g.w = 0; g.off = 0;
    d_lrec(L, m, n, g, out);
}
// start value alone (Eq. 27) as mantissa * 2^e, for pinning against lgamma / closed forms
extern "C" void orc_d_top(int l, int k, const long double* half, long double* mant, long* e2) {
    ld mm; long ee; top_value(l, k, half[0], half[1], mm, ee); *mant = mm; *e2 = ee;
}

// ------------------------------------------------------------------------------------------------------------
// Sampling tables exposed for the tests.
// sampling: 0 = MW (L rings x 2L-1), 1 = HEALPix(nside), 2 = MW quadrature grid of band-limit 2L (2L rings), w = q_u,
//           3 = MWSS (L+1 rings x 2L), 4 = DH (2L rings x 2L-1), 5 = GL (L rings x 2L-1),
//           6 = MWSS quadrature grid of band-limit 2L (2L+1 rings), w = q_u
// ------------------------------------------------------------------------------------------------------------
static RingSet make_rings(int sampling, int L, int nside) {
    if (sampling == 1) return rings_healpix(nside);
    if (sampling == 2) {
        RingSet S = rings_mw(2 * L, 2 * L - 1);
        std::vector<ld> v; mw_theta_weights(2 * L, v);
        for (int u = 0; u < 2 * L; ++u) S.r[u].w = 2.0L * PI_L / (ld)(2 * L - 1) * v[u];
        return S;
    }
    if (sampling == 3) return rings_mwss(L, 2 * L);
    if (sampling == 4) return rings_dh(L);
    if (sampling == 5) return rings_gl(L);
    if (sampling == 6) {
        RingSet S = rings_mwss(2 * L, 2 * L);
        std::vector<ld> v; mwss_theta_weights(2 * L, v);
        for (int u = 0; u <= 2 * L; ++u) S.r[u].w = 2.0L * PI_L / (ld)(2 * L) * v[u];
        return S;
    }
    return rings_mw(L, 2 * L - 1);
}
static bool is_map_sampling(int sampling) { return sampling == 0 || sampling == 1 || sampling == 3 || sampling == 4 || sampling == 5; }
extern "C" int orc_num_rings(int sampling, int L, int nside) { return (int)make_rings(sampling, L, nside).r.size(); }
extern "C" long orc_num_pixels(int sampling, int L, int nside) { return make_rings(sampling, L, nside).npix; }
extern "C" void orc_ring_table(int sampling, int L, int nside, long double* cos_theta, long double* sin_theta,
                               int* nphi, long double* phi0, long double* weight, long* offset) {
    RingSet S = make_rings(sampling, L, nside);
    for (size_t i = 0; i < S.r.size(); ++i) {
        cos_theta[i] = S.r[i].ct; sin_theta[i] = S.r[i].st; nphi[i] = S.r[i].nphi; phi0[i] = S.r[i].phi0;
        weight[i] = S.r[i].w; offset[i] = S.r[i].off;
    }
}

// ------------------------------------------------------------------------------------------------------------
// theta-step building blocks (Eq. 30 / 33 with a d-function from provider T)
// ------------------------------------------------------------------------------------------------------------
static inline ld pref_s2(int l, int s) { return sgn_pow(s) * sqrtl((ld)(2 * l + 1) / (4.0L * PI_L)); }

// G_m(ring) = sum_l coef[l] * d^l_{m,n}(ring)   for one m, all rings in `sel`
static void theta_synth_column(int L, int m, int n, const RingSet& S, const std::vector<int>& sel,
                               const cld* coef /*[L]*/, cld* out /*[sel.size()]*/) {
    std::vector<ld> d(L);
    int l0 = abs(m) > abs(n) ? abs(m) : abs(n);
    for (size_t i = 0; i < sel.size(); ++i) {
        d_lrec(L, m, n, S.r[sel[i]], d.data());
        cld acc = {0, 0};
        for (int l = l0; l < L; ++l) { acc.re += coef[l].re * d[l]; acc.im += coef[l].im * d[l]; }
        out[i] = acc;
    }
}
// c[l] = sum_ring W[ring] * d^l_{m,n}(ring)   for one m (W already carries the quadrature weight)
static void theta_analyse_column(int L, int m, int n, const RingSet& S, const cld* W /*[nrings]*/, cld* out /*[L]*/) {
    std::vector<ld> d(L);
    for (int l = 0; l < L; ++l) out[l] = {0, 0};
    int l0 = abs(m) > abs(n) ? abs(m) : abs(n);
    for (size_t r = 0; r < S.r.size(); ++r) {
        d_lrec(L, m, n, S.r[r], d.data());
        for (int l = l0; l < L; ++l) { out[l].re += W[r].re * d[l]; out[l].im += W[r].im * d[l]; }
    }
}
// naive ring DFT, Eq. 31 without the weight:  F_m = sum_p f_p e^{-i m phi_p}
static cld ring_dft(const double* f /*complex interleaved, nphi*/, const Ring& g, int m) {
    cld ph = {cosl(-(ld)m * g.phi0), sinl(-(ld)m * g.phi0)};
    cld acc = {0, 0};
    for (int p = 0; p < g.nphi; ++p) {
        cld e = unit_root(-(long)m * p, g.nphi);
        cld v = {(ld)f[2 * p], (ld)f[2 * p + 1]};
        acc = cadd(acc, cmul(v, e));
    }
    return cmul(acc, ph);
}
// naive ring synthesis, Eq. 32:  f_p = sum_m F_m e^{i m phi_p},  m = -(L-1)..L-1, F indexed [m+L-1]
static void ring_synth(int L, const cld* F, const Ring& g, double* f /*complex interleaved*/) {
    std::vector<cld> Fp(2 * L - 1);
    for (int m = -(L - 1); m < L; ++m) {
        cld ph = {cosl((ld)m * g.phi0), sinl((ld)m * g.phi0)};
        Fp[m + L - 1] = cmul(F[m + L - 1], ph);
    }
    for (int p = 0; p < g.nphi; ++p) {
        cld acc = {0, 0};
        for (int m = -(L - 1); m < L; ++m) acc = cadd(acc, cmul(Fp[m + L - 1], unit_root((long)m * p, g.nphi)));
        f[2 * p] = (double)acc.re; f[2 * p + 1] = (double)acc.im;
    }
}
// MW forward steps (ii)-(iv) for one m: F_m on the L MW rings -> F_m on the 2L rings of MW(2L)
static void mw_upsample_column(int L, int m, int s, const cld* Fin /*[L]*/, cld* Fout /*[2L]*/) {
    int T = 2 * L - 1, T2 = 4 * L - 1;
    std::vector<cld> ext(T), Fmm(T);
    ld sg = sgn_pow(m + s);
    for (int t = 0; t < T; ++t) ext[t] = (t < L) ? Fin[t] : cscale(Fin[2 * L - 2 - t], sg);
    for (int mp = -(L - 1); mp < L; ++mp) {                 // F_{m m'} = (1/T) sum_t F_m(theta_t) e^{-i m' theta_t}
        cld acc = {0, 0};
        for (int t = 0; t < T; ++t) acc = cadd(acc, cmul(ext[t], unit_root_pi(-(long)mp * (2 * t + 1), T)));
        Fmm[mp + L - 1] = cscale(acc, 1.0L / (ld)T);
    }
    for (int u = 0; u < 2 * L; ++u) {                        // F_m(theta'_u) = sum_{m'} F_{m m'} e^{i m' theta'_u}
        cld acc = {0, 0};
        for (int mp = -(L - 1); mp < L; ++mp) acc = cadd(acc, cmul(Fmm[mp + L - 1], unit_root_pi((long)mp * (2 * u + 1), T2)));
        Fout[u] = acc;
    }
}

// MWSS forward steps (ii)-(iv) for one m: F_m on the L+1 MWSS rings -> F_m on the 2L+1 rings of MWSS(2L).
// The theta circle carries 2L samples theta_t = 2 pi t/(2L); the Nyquist bin m' = L is outside the band-limit and is dropped
// (reading R23 of DESIGN.md: "zero padding in the Fourier domain" of a signal band-limited at L keeps |m'| <= L-1).
static void mwss_upsample_column(int L, int m, int s, const cld* Fin /*[L+1]*/, cld* Fout /*[2L+1]*/) {
    int T = 2 * L, T2 = 4 * L;
    std::vector<cld> ext(T), Fmm(2 * L - 1);
    ld sg = sgn_pow(m + s);
    for (int t = 0; t < T; ++t) ext[t] = (t <= L) ? Fin[t] : cscale(Fin[2 * L - t], sg);
    for (int mp = -(L - 1); mp < L; ++mp) {                 // F_{m m'} = (1/T) sum_t F_m(theta_t) e^{-i m' theta_t}
        cld acc = {0, 0};
        for (int t = 0; t < T; ++t) acc = cadd(acc, cmul(ext[t], unit_root(-(long)mp * t, T)));
        Fmm[mp + L - 1] = cscale(acc, 1.0L / (ld)T);
    }
    for (int u = 0; u <= 2 * L; ++u) {                       // F_m(theta'_u) = sum_{m'} F_{m m'} e^{i m' theta'_u}, theta'_u = 2 pi u/(4L)
        cld acc = {0, 0};
        for (int mp = -(L - 1); mp < L; ++mp) acc = cadd(acc, cmul(Fmm[mp + L - 1], unit_root((long)mp * u, T2)));
        Fout[u] = acc;
    }
}

// ------------------------------------------------------------------------------------------------------------
// S^2 transforms.  Layouts (row-major, complex = interleaved doubles):
//   flm[L][2L-1], column m+L-1;  MW map f[L][2L-1];  HEALPix map f[12 nside^2] ring-ordered.
// ------------------------------------------------------------------------------------------------------------
// inverse on a subset of rings: out = the selected rings' samples, concatenated in `ring_idx` order.
extern "C" int orc_s2_inverse_rings(int L, int spin, int sampling, int nside, const double* flm,
                                    int nsel, const int* ring_idx, double* f_out) {
    if (L < 1 || abs(spin) >= L || !is_map_sampling(sampling)) return 1;
    RingSet S = make_rings(sampling, L, nside);
    std::vector<int> sel(ring_idx, ring_idx + nsel);
    for (int i : sel) if (i < 0 || i >= (int)S.r.size()) return 1;
    int M = 2 * L - 1;
    std::vector<cld> F((size_t)M * nsel);           // [m][sel]
#pragma omp parallel for schedule(dynamic, 1)
    for (int mi = 0; mi < M; ++mi) {
        int m = mi - (L - 1);
        std::vector<cld> coef(L);
        for (int l = 0; l < L; ++l) {
            ld p = (l >= abs(spin) && l >= abs(m)) ? pref_s2(l, spin) : 0.0L;
            coef[l] = {p * (ld)flm[2 * ((size_t)l * M + mi)], p * (ld)flm[2 * ((size_t)l * M + mi) + 1]};
        }
        theta_synth_column(L, m, -spin, S, sel, coef.data(), &F[(size_t)mi * nsel]);
    }
    std::vector<long> ooff(nsel + 1, 0);
    for (int i = 0; i < nsel; ++i) ooff[i + 1] = ooff[i] + S.r[sel[i]].nphi;
#pragma omp parallel for schedule(dynamic, 1)
    for (int i = 0; i < nsel; ++i) {
        std::vector<cld> Fr(M);
        for (int mi = 0; mi < M; ++mi) Fr[mi] = F[(size_t)mi * nsel + i];
        ring_synth(L, Fr.data(), S.r[sel[i]], f_out + 2 * ooff[i]);
    }
    return 0;
}
extern "C" int orc_s2_inverse(int L, int spin, int sampling, int nside, const double* flm, double* f) {
    int nr = orc_num_rings(sampling, L, nside);
    std::vector<int> all(nr); for (int i = 0; i < nr; ++i) all[i] = i;
    return orc_s2_inverse_rings(L, spin, sampling, nside, flm, nr, all.data(), f);
}
// forward on a subset of harmonic orders: out[nsel][L] complex, row i = all l for m = m_list[i].
extern "C" int orc_s2_forward_columns(int L, int spin, int sampling, int nside, const double* f,
                                      int nsel, const int* m_list, double* flm_cols) {
    if (L < 1 || abs(spin) >= L || !is_map_sampling(sampling)) return 1;
    RingSet S = make_rings(sampling, L, nside);
    // rings the theta-quadrature runs on: the upsampled grids for MW / MWSS, the sample rings themselves otherwise
    RingSet Q = (sampling == 0) ? make_rings(2, L, nside) : (sampling == 3) ? make_rings(6, L, nside) : S;
    int nr = (int)S.r.size(), nq = (int)Q.r.size();
    for (int i = 0; i < nsel; ++i) if (abs(m_list[i]) >= L) return 1;
#pragma omp parallel for schedule(dynamic, 1)
    for (int i = 0; i < nsel; ++i) {
        int m = m_list[i];
        std::vector<cld> Fm(nr), W(nq), out(L);
        for (int r = 0; r < nr; ++r) Fm[r] = ring_dft(f + 2 * S.r[r].off, S.r[r], m);            // Eq. 31 (weight applied below)
        if (sampling == 0) mw_upsample_column(L, m, spin, Fm.data(), W.data());
        else if (sampling == 3) mwss_upsample_column(L, m, spin, Fm.data(), W.data());
        else W = Fm;
        for (int r = 0; r < nq; ++r) W[r] = cscale(W[r], Q.r[r].w);
        theta_analyse_column(L, m, -spin, Q, W.data(), out.data());                               // Eq. 30
        for (int l = 0; l < L; ++l) {
            ld p = (l >= abs(spin) && l >= abs(m)) ? pref_s2(l, spin) : 0.0L;
            flm_cols[2 * ((size_t)i * L + l)] = (double)(p * out[l].re);
            flm_cols[2 * ((size_t)i * L + l) + 1] = (double)(p * out[l].im);
        }
    }
    return 0;
}
extern "C" int orc_s2_forward(int L, int spin, int sampling, int nside, const double* f, double* flm) {
    int M = 2 * L - 1;
    std::vector<int> ms(M); for (int i = 0; i < M; ++i) ms[i] = i - (L - 1);
    std::vector<double> cols((size_t)2 * M * L);
    int rc = orc_s2_forward_columns(L, spin, sampling, nside, f, M, ms.data(), cols.data());
    if (rc) return rc;
    for (int mi = 0; mi < M; ++mi) for (int l = 0; l < L; ++l) {
        flm[2 * ((size_t)l * M + mi)] = cols[2 * ((size_t)mi * L + l)];
        flm[2 * ((size_t)l * M + mi) + 1] = cols[2 * ((size_t)mi * L + l) + 1];
    }
    return 0;
}
// theta-step only (Eq. 33): F[m_sel][ring] for selected m, all rings of the sampling -- used to check the GPU
// kernel's F_m(theta) directly at sizes where the full map is too expensive (L = 8192, "columns mode").
extern "C" int orc_s2_theta_inverse_columns(int L, int spin, int sampling, int nside, const double* flm,
                                            int nsel, const int* m_list, double* F_cols) {
    if (L < 1 || abs(spin) >= L || sampling < 0 || sampling > 6) return 1;
    RingSet S = make_rings(sampling, L, nside);
    int nr = (int)S.r.size(), M = 2 * L - 1;
    std::vector<int> all(nr); for (int i = 0; i < nr; ++i) all[i] = i;
#pragma omp parallel for schedule(dynamic, 1)
    for (int i = 0; i < nsel; ++i) {
        int m = m_list[i], mi = m + L - 1;
        std::vector<cld> coef(L), out(nr);
        for (int l = 0; l < L; ++l) {
            ld p = (l >= abs(spin) && l >= abs(m)) ? pref_s2(l, spin) : 0.0L;
            coef[l] = {p * (ld)flm[2 * ((size_t)l * M + mi)], p * (ld)flm[2 * ((size_t)l * M + mi) + 1]};
        }
        theta_synth_column(L, m, -spin, S, all, coef.data(), out.data());
        for (int r = 0; r < nr; ++r) { F_cols[2 * ((size_t)i * nr + r)] = (double)out[r].re; F_cols[2 * ((size_t)i * nr + r) + 1] = (double)out[r].im; }
    }
    return 0;
}

// theta-step only (Eq. 30): flm[:, m] = pref(l) sum_ring W[m_sel][ring] d^l_{m,-s}(theta_ring) for selected m on the rings of
// `sampling` (any code of make_rings, incl. the quadrature grids 2 and 6); W already carries the quadrature weight.
// out[nsel][L].  Used to check the GPU theta-forward entry point and as the timed sample of the CPU baseline.
extern "C" int orc_s2_theta_forward_columns(int L, int spin, int sampling, int nside, const double* W_cols,
                                            int nsel, const int* m_list, double* flm_cols) {
    if (L < 1 || abs(spin) >= L || sampling < 0 || sampling > 6) return 1;
    RingSet S = make_rings(sampling, L, nside);
    int nr = (int)S.r.size();
    for (int i = 0; i < nsel; ++i) if (abs(m_list[i]) >= L) return 1;
#pragma omp parallel for schedule(dynamic, 1)
    for (int i = 0; i < nsel; ++i) {
        int m = m_list[i];
        std::vector<cld> W(nr), out(L);
        for (int r = 0; r < nr; ++r) W[r] = {(ld)W_cols[2 * ((size_t)i * nr + r)], (ld)W_cols[2 * ((size_t)i * nr + r) + 1]};
        theta_analyse_column(L, m, -spin, S, W.data(), out.data());
        for (int l = 0; l < L; ++l) {
            ld p = (l >= abs(spin) && l >= abs(m)) ? pref_s2(l, spin) : 0.0L;
            flm_cols[2 * ((size_t)i * L + l)] = (double)(p * out[l].re);
            flm_cols[2 * ((size_t)i * L + l) + 1] = (double)(p * out[l].im);
        }
    }
    return 0;
}

// ------------------------------------------------------------------------------------------------------------
// Adjoints (Sec. 5.3): conjugate transposes of the two linear maps above, as plain sums.
// ------------------------------------------------------------------------------------------------------------
// (F^-1)^H, Eq. 56-58: the inverse transform is f = sum_lm flm sY_lm on the sample rings, so its adjoint is
//   flm = sum_{theta,phi} conj(sY_lm(theta,phi)) f(theta,phi)
// -- the analysis sum on the SAMPLE rings without quadrature weights (F Q^-1 of Eq. 58 where a direct quadrature exists).
// Selected harmonic orders; out[nsel][L].
extern "C" int orc_s2_inverse_adjoint_columns(int L, int spin, int sampling, int nside, const double* f,
                                              int nsel, const int* m_list, double* flm_cols) {
    if (L < 1 || abs(spin) >= L || !is_map_sampling(sampling)) return 1;
    RingSet S = make_rings(sampling, L, nside);
    int nr = (int)S.r.size();
    for (int i = 0; i < nsel; ++i) if (abs(m_list[i]) >= L) return 1;
#pragma omp parallel for schedule(dynamic, 1)
    for (int i = 0; i < nsel; ++i) {
        int m = m_list[i];
        std::vector<cld> Fm(nr), out(L);
        for (int r = 0; r < nr; ++r) Fm[r] = ring_dft(f + 2 * S.r[r].off, S.r[r], m);     // sum_p f e^{-i m phi_p}
        theta_analyse_column(L, m, -spin, S, Fm.data(), out.data());                     // sum_ring d^l_{m,-s} F_m
        for (int l = 0; l < L; ++l) {
            ld p = (l >= abs(spin) && l >= abs(m)) ? pref_s2(l, spin) : 0.0L;
            flm_cols[2 * ((size_t)i * L + l)] = (double)(p * out[l].re);
            flm_cols[2 * ((size_t)i * L + l) + 1] = (double)(p * out[l].im);
        }
    }
    return 0;
}
// F^H, Eq. 50-52.  Direct-quadrature samplings (HEALPix, DH, GL): F = Y^H Q, so F^H flm = Q (sum_lm flm sY_lm) -- Eq. 52 literally.
// MW / MWSS: the forward transform is the chain (i) phi-DFT, (ii) torus extension, (iii) theta-DFT, (iv) evaluation on the
// quadrature grid, (v) weights, (vi) Eq. 30; its adjoint is the conjugate-transposed chain in reverse order:
//   (vi,v)^H  G_m(theta'_u) = q_u sum_l pref(l) d^l_{m,-s}(theta'_u) flm
//   (iv)^H    A_{m m'}      = sum_u G_m(theta'_u) e^{-i m' theta'_u}
//   (iii)^H   X_m(theta_t)  = (1/T) sum_{m'} A_{m m'} e^{+i m' theta_t}          for every t of the theta circle
//   (ii)^H    F_m(theta_t)  = X_m(theta_t) + (-1)^{m+s} X_m(theta_reflect(t))     (rings that are their own reflection: X_m alone)
//   (i)^H     f(theta_t, phi_p) = sum_m F_m(theta_t) e^{+i m phi_p}
extern "C" int orc_s2_forward_adjoint(int L, int spin, int sampling, int nside, const double* flm, double* f) {
    if (L < 1 || abs(spin) >= L || !is_map_sampling(sampling)) return 1;
    RingSet S = make_rings(sampling, L, nside);
    bool up = (sampling == 0 || sampling == 3);
    RingSet Q = (sampling == 0) ? make_rings(2, L, nside) : (sampling == 3) ? make_rings(6, L, nside) : S;
    int nr = (int)S.r.size(), nq = (int)Q.r.size(), M = 2 * L - 1;
    std::vector<int> allq(nq); for (int i = 0; i < nq; ++i) allq[i] = i;
    std::vector<cld> F((size_t)M * nr);             // [m][sample ring]
#pragma omp parallel for schedule(dynamic, 1)
    for (int mi = 0; mi < M; ++mi) {
        int m = mi - (L - 1);
        std::vector<cld> coef(L), G(nq);
        for (int l = 0; l < L; ++l) {
            ld p = (l >= abs(spin) && l >= abs(m)) ? pref_s2(l, spin) : 0.0L;
            coef[l] = {p * (ld)flm[2 * ((size_t)l * M + mi)], p * (ld)flm[2 * ((size_t)l * M + mi) + 1]};
        }
        theta_synth_column(L, m, -spin, Q, allq, coef.data(), G.data());
        for (int u = 0; u < nq; ++u) G[u] = cscale(G[u], Q.r[u].w);
        if (!up) { for (int r = 0; r < nr; ++r) F[(size_t)mi * nr + r] = G[r]; continue; }
        // MW: T = 2L-1 circle samples theta_t = (2t+1)pi/T, quadrature grid theta'_u = (2u+1)pi/(4L-1);
        // MWSS: T = 2L circle samples theta_t = 2 pi t/T, quadrature grid theta'_u = 2 pi u/(4L).
        bool mw = sampling == 0;
        int T = mw ? 2 * L - 1 : 2 * L;
        std::vector<cld> A(2 * L - 1), X(T);
        for (int mp = -(L - 1); mp < L; ++mp) {
            cld acc = {0, 0};
            for (int u = 0; u < nq; ++u) {
                cld e = mw ? unit_root_pi(-(long)mp * (2 * u + 1), 4 * L - 1) : unit_root(-(long)mp * u, 4 * L);
                acc = cadd(acc, cmul(G[u], e));
            }
            A[mp + L - 1] = acc;
        }
        for (int t = 0; t < T; ++t) {
            cld acc = {0, 0};
            for (int mp = -(L - 1); mp < L; ++mp) {
                cld e = mw ? unit_root_pi((long)mp * (2 * t + 1), T) : unit_root((long)mp * t, T);
                acc = cadd(acc, cmul(A[mp + L - 1], e));
            }
            X[t] = cscale(acc, 1.0L / (ld)T);
        }
        ld sg = sgn_pow(m + spin);
        for (int t = 0; t < nr; ++t) {
            int tr = mw ? 2 * L - 2 - t : 2 * L - t;            // reflection of ring t on the theta circle
            bool self = mw ? (t == L - 1) : (t == 0 || t == L);
            F[(size_t)mi * nr + t] = self ? X[t] : cadd(X[t], cscale(X[tr], sg));
        }
    }
#pragma omp parallel for schedule(dynamic, 1)
    for (int r = 0; r < nr; ++r) {
        std::vector<cld> Fr(M);
        for (int mi = 0; mi < M; ++mi) Fr[mi] = F[(size_t)mi * nr + r];
        ring_synth(L, Fr.data(), S.r[r], f + 2 * S.r[r].off);
    }
    return 0;
}

// Un-separated definitions for tiny L (provider E, O(L^4)): Eq. 4 and Eq. 19 summed term by term.
extern "C" int orc_s2_inverse_direct(int L, int spin, int sampling, int nside, const double* flm, double* f) {
    if (L > 24) return 1;
    RingSet S = make_rings(sampling, L, nside); int M = 2 * L - 1;
    for (const Ring& g : S.r) for (int p = 0; p < g.nphi; ++p) {
        ld phi = g.phi0 + 2 * PI_L * (ld)p / (ld)g.nphi; cld acc = {0, 0};
        for (int l = abs(spin); l < L; ++l) for (int m = -l; m <= l; ++m) {
            ld y = pref_s2(l, spin) * d_explicit_hs(l, m, -spin, g.c2, g.s2);
            cld e = {cosl((ld)m * phi), sinl((ld)m * phi)};
            cld c = {(ld)flm[2 * ((size_t)l * M + m + L - 1)], (ld)flm[2 * ((size_t)l * M + m + L - 1) + 1]};
            acc = cadd(acc, cscale(cmul(c, e), y));
        }
        f[2 * (g.off + p)] = (double)acc.re; f[2 * (g.off + p) + 1] = (double)acc.im;
    }
    return 0;
}
// Eq. 19 with the ring set's own weights (HEALPix: 4pi/Npix).  Not defined for MW (its quadrature needs the
// upsampled grid), so sampling must be 1.
extern "C" int orc_s2_forward_direct(int L, int spin, int sampling, int nside, const double* f, double* flm) {
    if (L > 24 || sampling != 1) return 1;
    RingSet S = make_rings(sampling, L, nside); int M = 2 * L - 1;
    for (int i = 0; i < 2 * L * M; ++i) flm[i] = 0;
    for (int l = abs(spin); l < L; ++l) for (int m = -l; m <= l; ++m) {
        cld acc = {0, 0};
        for (const Ring& g : S.r) {
            ld y = pref_s2(l, spin) * d_explicit_hs(l, m, -spin, g.c2, g.s2);
            for (int p = 0; p < g.nphi; ++p) {
                ld phi = g.phi0 + 2 * PI_L * (ld)p / (ld)g.nphi;
                cld e = {cosl((ld)m * phi), -sinl((ld)m * phi)};
                cld v = {(ld)f[2 * (g.off + p)], (ld)f[2 * (g.off + p) + 1]};
                acc = cadd(acc, cscale(cmul(v, e), y * g.w));
            }
        }
        flm[2 * ((size_t)l * M + m + L - 1)] = (double)acc.re; flm[2 * ((size_t)l * M + m + L - 1) + 1] = (double)acc.im;
    }
    return 0;
}

// ------------------------------------------------------------------------------------------------------------
// SO(3) transforms on the MW-SO3 sampling: alpha_a = 2 pi a/(2L-1), beta_b = (2b+1)pi/(2L-1), gamma_g = 2 pi g/(2N-1)
// (PAPER.md:435-437).  f[2N-1][L][2L-1] = (gamma, beta, alpha);  flmn[2N-1][L][2L-1] = (n+N-1, l, m+L-1).
// ------------------------------------------------------------------------------------------------------------
extern "C" int orc_so3_inverse(int L, int N, const double* flmn, double* f) {
    if (L < 1 || N < 1 || N > L) return 1;
    RingSet S = rings_mw(L, 2 * L - 1);
    int M = 2 * L - 1, NG = 2 * N - 1;
    std::vector<int> all(L); for (int i = 0; i < L; ++i) all[i] = i;
    std::vector<cld> G((size_t)NG * M * L);                     // [n][m][beta] = sum_l (2l+1)/(8pi^2) flmn d^l_mn(beta)
#pragma omp parallel for schedule(dynamic, 1) collapse(2)
    for (int ni = 0; ni < NG; ++ni) for (int mi = 0; mi < M; ++mi) {
        int n = ni - (N - 1), m = mi - (L - 1);
        std::vector<cld> coef(L);
        for (int l = 0; l < L; ++l) {
            ld p = (l >= abs(n) && l >= abs(m)) ? (ld)(2 * l + 1) / (8.0L * PI_L * PI_L) : 0.0L;
            size_t idx = ((size_t)ni * L + l) * M + mi;
            coef[l] = {p * (ld)flmn[2 * idx], p * (ld)flmn[2 * idx + 1]};
        }
        theta_synth_column(L, m, n, S, all, coef.data(), &G[((size_t)ni * M + mi) * L]);
    }
    // f(alpha_a, beta_b, gamma_g) = sum_n e^{i n gamma_g} sum_m e^{i m alpha_a} G[n][m][b]       (Eq. 13 with Eq. 10)
#pragma omp parallel for schedule(dynamic, 1)
    for (int b = 0; b < L; ++b) {
        std::vector<cld> H((size_t)NG * M);                      // [n][a]
        for (int ni = 0; ni < NG; ++ni) for (int a = 0; a < M; ++a) {
            cld acc = {0, 0};
            for (int mi = 0; mi < M; ++mi) acc = cadd(acc, cmul(G[((size_t)ni * M + mi) * L + b], unit_root((long)(mi - (L - 1)) * a, M)));
            H[(size_t)ni * M + a] = acc;
        }
        for (int g = 0; g < NG; ++g) for (int a = 0; a < M; ++a) {
            cld acc = {0, 0};
            for (int ni = 0; ni < NG; ++ni) acc = cadd(acc, cmul(H[(size_t)ni * M + a], unit_root((long)(ni - (N - 1)) * g, NG)));
            size_t idx = ((size_t)g * L + b) * M + a;
            f[2 * idx] = (double)acc.re; f[2 * idx + 1] = (double)acc.im;
        }
    }
    return 0;
}
extern "C" int orc_so3_forward(int L, int N, const double* f, double* flmn) {
    if (L < 1 || N < 1 || N > L) return 1;
    RingSet Q = make_rings(2, L, 0);                             // MW(2L) beta grid, w = (2pi/(2L-1)) v_u
    int M = 2 * L - 1, NG = 2 * N - 1;
    // (a) f_n(alpha,beta) = (2pi/(2N-1)) sum_g f e^{-i n gamma_g}   (Eq. 16 discretised)
    std::vector<cld> fn((size_t)NG * L * M);
#pragma omp parallel for schedule(static)
    for (int b = 0; b < L; ++b) for (int a = 0; a < M; ++a) for (int ni = 0; ni < NG; ++ni) {
        cld acc = {0, 0};
        for (int g = 0; g < NG; ++g) {
            size_t idx = ((size_t)g * L + b) * M + a;
            cld v = {(ld)f[2 * idx], (ld)f[2 * idx + 1]};
            acc = cadd(acc, cmul(v, unit_root(-(long)(ni - (N - 1)) * g, NG)));
        }
        fn[((size_t)ni * L + b) * M + a] = cscale(acc, 2.0L * PI_L / (ld)NG);
    }
#pragma omp parallel for schedule(dynamic, 1) collapse(2)
    for (int ni = 0; ni < NG; ++ni) for (int mi = 0; mi < M; ++mi) {
        int n = ni - (N - 1), m = mi - (L - 1);
        std::vector<cld> Fm(L), W(2 * L), out(L);
        for (int b = 0; b < L; ++b) {                            // (b) alpha DFT
            cld acc = {0, 0};
            for (int a = 0; a < M; ++a) acc = cadd(acc, cmul(fn[((size_t)ni * L + b) * M + a], unit_root(-(long)m * a, M)));
            Fm[b] = acc;
        }
        mw_upsample_column(L, m, -n, Fm.data(), W.data());       // (c),(d): extension sign (-1)^{m-n}
        for (int u = 0; u < 2 * L; ++u) W[u] = cscale(W[u], Q.r[u].w);
        theta_analyse_column(L, m, n, Q, W.data(), out.data());  // (e) sum_u q_u d^l_mn(beta'_u) F(beta'_u)   (Eq. 20)
        for (int l = 0; l < L; ++l) {
            bool ok = (l >= abs(n) && l >= abs(m));
            size_t idx = ((size_t)ni * L + l) * M + mi;
            flmn[2 * idx] = ok ? (double)out[l].re : 0.0; flmn[2 * idx + 1] = ok ? (double)out[l].im : 0.0;
        }
    }
    return 0;
}

extern "C" int orc_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
extern "C" void orc_set_threads(int n) {
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}
