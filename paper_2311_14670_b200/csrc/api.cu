// api.cu -- the C ABI of include/b200sht.h: plans, workspace layout, stage orchestration, cuFFT calls.
//
// Data flow; everything is m-major so that the hot kernels read contiguous tiles:
//   inverse:  coef[l][m] --prep--> G[pass][m][l]  ==theta_inverse==>  F[m mod NB][ring]  --cuFFT(phi)--> map
//   forward:  map --cuFFT(phi)--> Fa[m][ring] --MW extend / theta-FFT / pad / theta-iFFT--> U[m][ring']
//             --weight_split--> W[pass][m][ring']  ==theta_forward==>  H[m][l]  --finalize--> coef[l][m]
#include "../../include/b200sht.h"
#include "internal.h"
#include "staging.h"

#include <cufft.h>
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <map>
#include <mutex>
#include <string>
#include <tuple>
#include <vector>

namespace {

thread_local long g_launches = 0;
thread_local double g_bytes = 0;      // algorithmic bytes enqueued since the last timed-section boundary (count_bytes)
thread_local std::string g_err;

typedef long double ld;
const ld PI_L = 3.14159265358979323846264338327950288L;

inline size_t rup(size_t x, size_t a) { return (x + a - 1) / a * a; }

#define CK(call)                                                                                   \
    do {                                                                                           \
        cudaError_t e__ = (call);                                                                  \
        if (e__ != cudaSuccess) {                                                                  \
            g_err = std::string(#call) + ": " + cudaGetErrorString(e__);                           \
            return SHT_ECUDA;                                                                      \
        }                                                                                          \
    } while (0)
#define CF(call)                                                                                   \
    do {                                                                                           \
        cufftResult r__ = (call);                                                                  \
        if (r__ != CUFFT_SUCCESS) {                                                                \
            g_err = std::string(#call) + ": cufft error " + std::to_string((int)r__);              \
            return SHT_ECUFFT;                                                                     \
        }                                                                                          \
    } while (0)
#define CS(call)                                                                                   \
    do {                                                                                           \
        sht_status s__ = (call);                                                                   \
        if (s__ != SHT_OK) return s__;                                                             \
    } while (0)

// ---- one set of iso-latitude rings the theta kernels run on -----------------------------------------------------
struct RingSet {
    int nth = 0, ntp = 0;      // regular rings, padded count (multiple of 128; > nth so a pole ring fits)
    bool pole = false;         // a theta = pi ring right after the regular rings (MW, MWSS; Eq. 29)
    bool pole_n = false;       // a theta = 0 ring in front of the regular rings (MWSS; Eq. 28)
    bool symmetric = false;    // ring nth-1-t is the mirror image pi - theta_t of ring t
    int nfull = 0;             // > 0: this set is the northern half (incl. an equator ring) of a symmetric set of nfull rings
    std::vector<ld> ct, c2, s2;  // host: cos(theta), cos(theta/2), sin(theta/2) of the regular rings
    double *csc = nullptr, *tau = nullptr, *sig = nullptr, *c2hi = nullptr, *c2lo = nullptr, *s2hi = nullptr, *s2lo = nullptr;
    double* wq = nullptr;      // [ntp] forward quadrature weight per ring (incl. the pole ring at index nth)
    struct Start { double* val; uint8_t* k; };
    std::map<int, Start> start;   // second index n -> windowed start values [Lp][ntp]
    std::map<int, int*> mlo;      // key 2n (pass A) / 2n+1 (pass B) -> per-ring first served step
};

struct PassHost {
    ThetaPass p;
    int mode;                  // 0 PM, 1 P
};

enum { CAT_HOT = 0, CAT_FFT = 1, CAT_STAGE = 2 };
// internal samplings of the adjoint helper plans: the rings of an MW / MWSS map with a direct, unit-weight "quadrature"
enum { SHT_INT_MWRINGS = 100, SHT_INT_MWSSRINGS = 101 };

}  // namespace

struct sht_plan {
    int kind = 0;              // 0 S^2, 1 SO(3)
    int L = 0, spin = 0, sampling = 0, nside = 0, reality = 0, N = 1;
    int Lp = 0, NB = 0;        // padded L; number of phi bins = rows of F / Fa / Z = length of the phi FFT (2L-1; MWSS: 2L)
    int M = 0;                 // 2L-1: row length of the coefficient arrays flm[L][M]
    int nrmap = 0;             // rings of the map (equiangular samplings): L (MW, GL), L+1 (MWSS), 2L (DH)
    size_t map_elems = 0;      // samples of one map
    int Tcirc = 0;             // MW / MWSS: samples of the theta circle the forward extension works on (= NB)
    int col0 = 0;              // column of F (= ring of the map) of the first regular ring of the inverse ring set (MWSS: 1)
    std::vector<ld> gl_w;      // GL: Gauss weights of the rings
    int nslab = 1;             // number of second-index values (1 for S^2, 2N-1 for SO(3), in gamma-FFT bin order)
    bool f32_inner = false;    // set while an fp32 transform runs its fp64-array core
    int dtype = SHT_F64;       // arithmetic of the hot kernels.  SHT_F32: fp32 kernels (theta_f32.cu); staging and FFTs stay fp64
    bool io_f32 = false;       // the public arrays are fp32 (plan created with SHT_F32): fp64 copies around the core.  spin != 0 plans created
                               // with SHT_F32 have io_f32 with dtype == SHT_F64 (the fp32 kernels recurse the second index n = 0 only)
    float4* ab32 = nullptr;    // fp32: [L][Lp] recursion coefficients {A, A, -B, -B}
    float *lam32_inv = nullptr, *lam32_fwd = nullptr;
    float *st32_inv = nullptr, *st32_fwd = nullptr; uint16_t *k16_inv = nullptr, *k16_fwd = nullptr;   // fp32 start values
    double2 *io_a = nullptr, *io_b = nullptr;   // fp32: fp64 copies of the public arrays
    int invsym = 0;            // MW spin-0 inverse: F_m on the L midpoint rings (north-south fold), then FFT resampling to the MW rings
    cufftHandle fft_sym = 0;   // length 2L, batch 2L-1
    int fold0i = 0;            // spin-0 plans on ring sets symmetric about the equator (HEALPix): the inverse recursion too
    int F_ld = 0, F_nrings = 0;   // row length of F[bin][F_ld] and the number of rings it holds (incl. a pole ring)
    bool upsampled = false;    // MW / MWSS: the forward transform extends F_m to the theta circle and upsamples to the quadrature rings
    // silent-head skip tables (ThetaArgs::skip_*): [direction 0 inverse / 1 forward][kernel mode 0 PM / 1 P]
    bool skip = false, skip_ready = false;
    int* skip_p0[2][2] = {{nullptr, nullptr}, {nullptr, nullptr}};
    double* skip_state[2][2] = {{nullptr, nullptr}, {nullptr, nullptr}};
    int skip_nb[2][2] = {{0, 0}, {0, 0}};
    double skip_pairs[2] = {0, 0}, all_pairs[2] = {0, 0};     // block-pairs skipped / in total, per direction (sht_plan_skip_fraction)
    bool inv_fold = false;     // n != 0 S^2 plans: the inverse runs ONE fold pass (+m at a ring, -m at its mirror ring) where its rings are symmetric
    int pair = 0;              // MW / MWSS: the theta-circle FFTs carry two orders m per column (staging.cu u_get): prow = L rows instead of NB
    int prow = 0;              // rows of the theta-circle arrays X / Z the upsampling (and the symmetric-ring resampling) works on
    int fold0 = 0;             // spin-0 S^2 plans: the forward recursion runs on the northern quadrature rings only
    bool precomp = false;      // SHT_OPT_PRECOMPUTE: stored d-function tables (precompute.cu, Sec. 4.3)
    int shard_rank = 0, shard_n = 1;   // ring shard (sht_plan_set_shard): this plan serves share shard_rank of shard_n of the kernel rings
    unsigned opts = 0;         // SHT_OPT_* given at creation
    // Helper plans of the adjoint entry points (SHT_OPT_ADJOINT; MW / MWSS only, where the forward quadrature does not run on the
    // rings of the map): adj_inv runs the FORWARD-type kernel on the rings of the map ((F^-1)^H, Eq. 58), adj_fwd runs the
    // INVERSE-type kernel on the 2L quadrature rings (F^H, Eq. 52).  A helper owns only the tables / buffers of its one direction.
    sht_plan *adj_inv = nullptr, *adj_fwd = nullptr;
    // SO(3) plans with SHT_OPT_ADJOINT: one S^2 adjoint plan per order n (spin -n), the l-scalings between the Wigner and the spin
    // normalisations (for even n; odd n flips the sign), one coefficient slab of scratch
    std::vector<sht_plan*> sub;
    double *so3_dfwd = nullptr, *so3_dinv = nullptr;
    double2* adj_tmp = nullptr;
    bool helper = false;
    int only_dir = 0;          // helper plans: 1 = inverse-type kernel only, 2 = forward-type kernel only
    double *it_map = nullptr, *it_coef = nullptr;   // HEALPix iterative refinement: residual map / coefficient update scratch
    double *it_f = nullptr, *it_acc = nullptr;      // ... of plans with fp32 public arrays: fp64 copies of the map and of the running coefficients
    double* wq_map = nullptr;  // [F_ld] quadrature weight of every ring of the map (direct-quadrature samplings; adjoints)
    double* wq_quad = nullptr; // [4L] MW / MWSS: weight of every one of the 2L quadrature rings (not folded; adjoints)
    int device = 0, nsm = 0;   // device the plan was created on and its SM count (tile choice)
    // CUDA graphs (launch-bound sizes): a whole transform is captured once per (direction, input, output) and replayed with one launch
    struct GraphEntry { int kind; const void* in; void* out; cudaGraphExec_t exec; long launches; };
    std::vector<GraphEntry> graphs;
    cudaStream_t cap_stream = nullptr;   // capture stream (the caller's stream may be the legacy default stream, which cannot capture)
    bool use_graph = false;
    int graph_hits = 0, graph_misses = 0;
    int* d_flag = nullptr;     // device flag raised by table kernels (start value outside the window-counter range)
    double sec_bytes[3] = {0, 0, 0};   // algorithmic bytes moved by the FFT / staging sections of the last transform (stage timing)
    int batch = 1;             // > 1: a batch of S^2 maps sharing one recursion (theta_mma.cu); then nslab = batch
    int loop = 1;              // > 1: a batch on a sampling / dtype without the batched kernels: the single-map plan runs map by map
    int ncg = 0, ncg_fwd = 0;  // batched path: column groups of 16 complex columns (inverse / forward passes)
    double* Ob = nullptr;      // batched path: result scratch of all passes
    std::vector<size_t> ob_off_inv, ob_off_fwd;   // per-pass offsets (doubles) into Ob
    std::vector<int> slab_n;   // second index n of d^l_{m,n} per slab
    int *d_slab_n = nullptr, *d_cslab = nullptr;   // device copies: n per slab; slab -> slab of the public coefficient array
    RingSet inv, fwd;          // rings of the inverse theta step / of the forward quadrature
    int kmin = 0, kstride = 0, krows = 0;
    int8_t* kexp = nullptr;
    double* rsq = nullptr;
    int mmin = 0, sgstride = 0;    // lowest recursion step of any pass; columns of the (s, G) table
    double* ctab = nullptr;        // [L - mmin][Lp] c_m(l)
    double2* sgtab = nullptr;      // [Lp/TQ][sgstride]
    double *scale_inv = nullptr, *scale_fwd = nullptr;   // [Lp] l-dependent factors
    // pass lists (host copies + device arrays), split by kernel mode
    std::vector<PassHost> pinv, pfwd;
    ThetaPass *d_inv_pm = nullptr, *d_inv_p = nullptr, *d_fwd_pm = nullptr, *d_fwd_p = nullptr;
    int n_inv_pm = 0, n_inv_p = 0, n_fwd_pm = 0, n_fwd_p = 0;
    // scratch
    double2 *F = nullptr, *Fa = nullptr, *X = nullptr, *Z = nullptr, *H = nullptr, *cplx = nullptr, *fn = nullptr;
    double2* polev = nullptr;  // [nslab] pole-ring values of the inverse
    double* tmp = nullptr;     // [2*Lp] plan-time scratch
    double* unit_wq = nullptr; // [fwd.ntp] ones (theta-stage entry point takes already weighted rows)
    size_t F_slab = 0, Fa_slab = 0, X_slab = 0, Z_slab = 0, H_slab = 0;
    int Ltp = 0;               // padded ring count of Fa rows
    int fwd_ld = 0;            // row length of the forward ring-sample array U (MW: 4L, HEALPix: padded ring count)
    // HEALPix ring-FFT staging (healpix.cu): Bluestein batch C[2(nside-1)][M], chirp spectra BF[nside-1][M], belt rows E
    int hp_M = 0, hp_ncap = 0, hp_neq = 0; long long hp_off_eq = 0;
    double2 *hp_C = nullptr, *hp_BF = nullptr, *hp_E = nullptr;
    cufftHandle fft_hp_cap = 0, fft_hp_eq = 0;
    void* fft_work = nullptr; size_t fft_work_bytes = 0;
    cufftHandle fft_phi_inv = 0, fft_phi_fwd = 0, fft_th1 = 0, fft_th2 = 0, fft_gamma = 0;
    // host-buffer calls (s2_*_host): ring FFTs in `nchunk` ring chunks, so that the PCIe copy of chunk k+1 overlaps the FFT of chunk k
    cufftHandle fft_phi_inv_c = 0, fft_phi_fwd_c = 0; int nchunk = 0;
    cudaStream_t copy_stream = nullptr; cudaEvent_t ev_copy[8] = {}, ev_begin = nullptr;
    bool skip_phi = false;     // set while a host-buffer call runs the ring FFT stage itself
    cufftHandle fft_alpha = 0; // SO(3): the ring FFTs of all (gamma / n, beta) rows in ONE batch, on the [slab][ring][phi] layout
    bool have_fft = false;
    std::map<cufftHandle, double> fft_elems;   // complex elements one execution of each handle transforms (byte accounting)
    // workspace
    void* work = nullptr; size_t work_bytes = 0, need_bytes = 0;
    bool ready = false;
    // timing
    bool timing = false;
    std::vector<cudaEvent_t> ev; std::vector<int> ev_cat; int ev_n = 0;
    double dsteps_inv = 0, dsteps_fwd = 0, flops_inv = 0, flops_fwd = 0;
};

namespace {

// ---- host-side ring geometry (long double; the GPU tables are split into hi/lo doubles where it matters) ---------
void rings_mw(RingSet& R, int Lt) {      // Eq. 37: theta_t = (2t+1)pi/(2Lt-1); ring Lt-1 is theta = pi
    R.nth = Lt - 1; R.pole = true;
    R.ct.resize(R.nth); R.c2.resize(R.nth); R.s2.resize(R.nth);
    for (int t = 0; t < R.nth; ++t) {
        ld th = PI_L * (ld)(2 * t + 1) / (ld)(2 * Lt - 1);
        R.ct[t] = cosl(th); R.c2[t] = cosl(th / 2); R.s2[t] = sinl(th / 2);
    }
    R.ntp = (int)rup((size_t)R.nth + 1, 128);
}

// Forward quadrature rings of the MW transform (R9): theta'_u = (2u+1)pi/(4L), u = 0..2L-1 -- the midpoints of
// 4L equispaced samples of the theta circle.  The paper upsamples F_m(theta) to "2L" rings; any ring set
// on which the quadrature of the band-limit-(2L-2) integrand is exact gives the same result, and this one has a
// power-of-two FFT length 4L (the MW(2L) set needs 4L-1, often prime) and no pole ring.
void rings_mid(RingSet& R, int nrings) {      // theta_u = (2u+1) pi / (2 nrings), u = 0..nrings-1
    R.nth = nrings; R.pole = false; R.symmetric = true;
    R.ct.resize(R.nth); R.c2.resize(R.nth); R.s2.resize(R.nth);
    for (int u = 0; u < R.nth; ++u) {
        ld th = PI_L * (ld)(2 * u + 1) / (ld)(2 * nrings);
        R.ct[u] = cosl(th); R.c2[u] = cosl(th / 2); R.s2[u] = sinl(th / 2);
    }
    R.ntp = (int)rup((size_t)R.nth, 128);
}

// MWSS, Eq. 39: theta_t = 2 pi t/(2L), t = 0..L.  Rings t = 0 and t = L are the poles (Eq. 28 / 29, handled apart);
// the regular rings t = 1..L-1 are symmetric about the equator.
void rings_mwss(RingSet& R, int L) {
    R.nth = L - 1; R.pole = true; R.pole_n = true; R.symmetric = true;
    R.ct.resize(R.nth); R.c2.resize(R.nth); R.s2.resize(R.nth);
    for (int i = 0; i < R.nth; ++i) {
        // mirror pairs get exactly mirrored trigonometry: evaluate on the northern ring
        const int t = i + 1, tn = t <= L - t ? t : L - t;
        ld th = PI_L * (ld)tn / (ld)L;
        ld c = cosl(th), c2 = cosl(th / 2), s2 = sinl(th / 2);
        if (2 * t == L) c = 0;
        const bool south = t > L - t;
        R.ct[i] = south ? -c : c; R.c2[i] = south ? s2 : c2; R.s2[i] = south ? c2 : s2;
    }
    R.ntp = (int)rup((size_t)R.nth + 2, 128);
}
// Gauss-Legendre rings: theta_t = acos(x_t), x_t the roots of P_L, north to south.  Newton's iteration in theta on
// P_L(cos theta) (three-term recurrence in long double), so the half angles keep full relative accuracy near the poles.  Also
// returns the Gauss weights 2/((1-x^2) P_L'(x)^2) (the weight Eq. 46 stands for, R22).
void rings_gl(RingSet& R, int L, std::vector<ld>* wts) {
    R.nth = L; R.pole = false; R.symmetric = true;
    R.ct.resize(L); R.c2.resize(L); R.s2.resize(L);
    if (wts) wts->assign(L, 0);
    auto pl = [L](ld x, ld& p, ld& dp) {
        ld p0 = 1, p1 = x;
        for (int k = 2; k <= L; ++k) { ld pk = ((ld)(2 * k - 1) * x * p1 - (ld)(k - 1) * p0) / (ld)k; p0 = p1; p1 = pk; }
        p = p1; dp = (ld)L * (x * p1 - p0) / (x * x - 1);
    };
    for (int t = 0; t < (L + 1) / 2; ++t) {
        ld th = PI_L * ((ld)t + 0.75L) / ((ld)L + 0.5L), p, dp;
        for (int it = 0; it < 100; ++it) {
            pl(cosl(th), p, dp);
            ld dth = p / (sinl(th) * dp);
            th += dth;
            if (fabsl(dth) < 1e-19L * th) break;
        }
        const bool eq = 2 * t + 1 == L;
        if (eq) th = PI_L / 2;
        pl(cosl(th), p, dp);
        const ld c = eq ? 0.0L : cosl(th), sn = eq ? 1.0L : sinl(th), c2 = cosl(th / 2), s2 = sinl(th / 2);
        const ld w = 2.0L / (sn * sn * dp * dp);
        R.ct[t] = c; R.c2[t] = c2; R.s2[t] = s2;
        R.ct[L - 1 - t] = -c; R.c2[L - 1 - t] = s2; R.s2[L - 1 - t] = c2;       // the mirror ring, exactly mirrored
        if (wts) { (*wts)[t] = w; (*wts)[L - 1 - t] = w; }
    }
    R.ntp = (int)rup((size_t)R.nth + 1, 128);
}

// HEALPix rings r = 1..4 nside-1 (public ring scheme, R11); half-angle trigonometry from z
void rings_healpix(RingSet& R, int nside) {
    R.nth = 4 * nside - 1; R.pole = false; R.symmetric = true;
    R.ct.resize(R.nth); R.c2.resize(R.nth); R.s2.resize(R.nth);
    const ld ns = (ld)nside;
    for (int i = 0; i < R.nth; ++i) {
        int r = i + 1, rr = r <= 2 * nside ? r : 4 * nside - r;
        ld z = rr < nside ? 1.0L - (ld)rr * (ld)rr / (3.0L * ns * ns) : 4.0L / 3.0L - 2.0L * (ld)rr / (3.0L * ns);
        if (r == 2 * nside) z = 0;
        if (r > 2 * nside) z = -z;
        R.ct[i] = z; R.c2[i] = sqrtl((1 + z) / 2); R.s2[i] = sqrtl((1 - z) / 2);
    }
    R.ntp = (int)rup((size_t)R.nth + 1, 128);
}

// keep the northern half of a symmetric ring set (n = 0 forward fold, theta_kernels.cu FOLD); ring t mirrors ring nfull-1-t
void north_only(RingSet& R) {
    R.nfull = R.nth; R.nth = (R.nth + 1) / 2; R.symmetric = false;
    R.ct.resize(R.nth); R.c2.resize(R.nth); R.s2.resize(R.nth);
    R.ntp = (int)rup((size_t)R.nth, 128);
}

struct Bump {
    size_t off = 0; char* base = nullptr;
    template <class T> T* take(size_t n) {
        off = rup(off, 256);
        T* p = base ? reinterpret_cast<T*>(base + off) : nullptr;
        off += n * sizeof(T);
        return p;
    }
};

// doubles of one pass's operand buffer (single-map kernels: rows m_end-1..L-1; batched: rows m_end..L-1 per column group)
size_t pass_in_doubles(const sht_plan* P, const PassHost& ph, bool fwd) {
    const size_t K = fwd ? P->fwd.ntp : P->Lp;
    if (P->batch > 1) return (size_t)(fwd ? P->ncg_fwd : P->ncg) * (P->L - ph.p.m_end) * K * (fwd && P->fold0 ? SHT_MMA_ROWF : SHT_MMA_ROW);
    const size_t rows = (size_t)(P->L - ph.p.m_end + 1);
    return fwd ? rows * K * (ph.mode == 0 ? 4 : 2) * (P->fold0 ? 2 : 1) : rows * K * theta_inverse_rowd(ph.mode);
}

void begin_transform(sht_plan* P) {
    P->ev_n = 0; g_bytes = 0;
    P->sec_bytes[0] = P->sec_bytes[1] = P->sec_bytes[2] = 0;
}
// Opens a timed section of category `cat` (and closes the previous one).  The algorithmic bytes the closed section moved (each
// array a staging kernel / FFT / memset reads or writes, once; counted by the launchers through count_bytes) are added to its
// category and reported by sht_plan_stage_bytes(), so that the HBM-bound stages can be quoted in GB/s.
void stage(sht_plan* P, int cat, cudaStream_t st) {
    if (!P->timing) { g_bytes = 0; return; }
    if (P->ev_n > 0) P->sec_bytes[P->ev_cat[P->ev_n - 1]] += g_bytes;     // bytes of the section this call closes
    g_bytes = 0;
    if (P->ev_n >= (int)P->ev.size()) return;
    cudaEventRecord(P->ev[P->ev_n], st);
    P->ev_cat[P->ev_n] = cat;
    P->ev_n++;
}

// Array dimensions that depend on the sampling (called once the ring sets and folds are fixed).
//   F  [slab][NB bins][F_ld]   F_m on the rings of the map (columns in map-ring order, poles included); Fa likewise (forward side)
//   X  [slab][NB bins][Tcirc]  MW / MWSS: F_m extended to the theta circle          Z [slab][NB][fwd_ld]: F_m on the quadrature rings
//   H  [slab][NB rows >= M][Lp]
void plan_dims(sht_plan* P) {
    const int L = P->L;
    P->M = 2 * L - 1;
    P->upsampled = P->sampling == SHT_MW || P->sampling == SHT_MWSS;
    switch (P->sampling) {
        case SHT_MWSS: case SHT_INT_MWSSRINGS: P->NB = 2 * L; P->nrmap = L + 1; break;
        case SHT_DH: P->NB = 2 * L - 1; P->nrmap = 2 * L; break;
        default: P->NB = 2 * L - 1; P->nrmap = L; break;         // MW, GL; HEALPix keeps 2L-1 "bins" as its F-row convention
    }
    P->Tcirc = P->NB;
    P->prow = P->pair ? L : P->NB;
    P->col0 = P->inv.pole_n ? 1 : 0;
    if (P->sampling == SHT_HEALPIX) {
        P->nrmap = 4 * P->nside - 1;
        P->map_elems = (size_t)12 * P->nside * P->nside;
    } else
        P->map_elems = (size_t)P->nrmap * P->NB;
    P->F_nrings = P->invsym ? L : P->nrmap;
    P->F_ld = (int)rup((size_t)P->F_nrings, 128);
    if (!P->inv.nfull && P->inv.ntp > P->F_ld) P->F_ld = P->inv.ntp;
    P->F_slab = (size_t)P->NB * P->F_ld;
    P->Ltp = P->F_ld;
    P->Fa_slab = (size_t)P->NB * P->Ltp;
    P->X_slab = (size_t)P->NB * P->Tcirc;
    const int nq = P->fwd.nfull ? P->fwd.nfull : P->fwd.nth;
    if (P->upsampled) P->fwd_ld = 4 * L;
    else if (P->sampling == SHT_HEALPIX) P->fwd_ld = (int)rup((size_t)nq + 1, 128);
    else P->fwd_ld = P->Ltp;                                       // DH / GL: the quadrature runs on the map's own rings (U = Fa)
    P->Z_slab = (size_t)P->NB * P->fwd_ld;
    P->H_slab = (size_t)P->NB * P->Lp;
}

// Walks the workspace layout.  With base == nullptr it only measures; otherwise it assigns every pointer.
void layout(sht_plan* P, char* base) {
    Bump B; B.base = base;
    const int L = P->L, Lp = P->Lp, NB = P->NB;
    P->d_flag = B.take<int>(64);
    P->d_slab_n = B.take<int>(P->nslab); P->d_cslab = B.take<int>(P->nslab);
    P->rsq = B.take<double>(2 * (size_t)Lp + 64);
    P->kexp = B.take<int8_t>((size_t)P->krows * P->kstride);
    P->ctab = B.take<double>((size_t)(L - P->mmin) * Lp);
    P->sgtab = B.take<double2>((size_t)P->krows * P->sgstride);
    P->scale_inv = B.take<double>(Lp);
    P->scale_fwd = B.take<double>(Lp);
    for (RingSet* R : {&P->inv, &P->fwd}) {
        if ((R == &P->inv && P->only_dir == 2) || (R == &P->fwd && P->only_dir == 1)) continue;
        R->csc = B.take<double>(R->ntp); R->tau = B.take<double>(R->ntp); R->sig = B.take<double>(R->ntp);
        R->c2hi = B.take<double>(R->ntp); R->c2lo = B.take<double>(R->ntp);
        R->s2hi = B.take<double>(R->ntp); R->s2lo = B.take<double>(R->ntp);
        R->wq = B.take<double>(R->ntp);
        for (auto& kv : R->start) {
            kv.second.val = B.take<double>((size_t)Lp * R->ntp);
            kv.second.k = B.take<uint8_t>((size_t)Lp * R->ntp);
        }
        for (auto& kv : R->mlo) kv.second = B.take<int>(R->ntp);
    }
    P->d_inv_pm = B.take<ThetaPass>(P->pinv.size() + 1); P->d_inv_p = B.take<ThetaPass>(P->pinv.size() + 1);
    P->d_fwd_pm = B.take<ThetaPass>(P->pfwd.size() + 1); P->d_fwd_p = B.take<ThetaPass>(P->pfwd.size() + 1);
    // per-pass operand buffers and lambda tables
    // (rows m = m_end-1 .. L-1; row m_end-1 is all zero: the dummy second step of a final odd pair reads it)
    for (auto& ph : P->pinv) {      // (empty for forward-only helpers, and vice versa)
        ph.p.in = B.take<double>(pass_in_doubles(P, ph, false));
        ph.p.lam = B.take<double>((size_t)(L - ph.p.m_end + 1) * P->inv.ntp);
    }
    for (auto& ph : P->pfwd) {
        ph.p.in = B.take<double>(pass_in_doubles(P, ph, true));
        ph.p.lam = B.take<double>((size_t)(L - ph.p.m_end + 1) * P->fwd.ntp);
    }
    if (P->skip) {           // per block of every fused launch: pairs to skip + the register state to start from
        for (int dir = 0; dir < 2; ++dir)
            for (int md = 0; md < 2; ++md) {
                const RingSet& R = dir ? P->fwd : P->inv;
                int np = 0;
                for (auto& ph : (dir ? P->pfwd : P->pinv)) np += ph.mode == md;
                P->skip_nb[dir][md] = 0;
                if (!np) continue;
                if (P->dtype == SHT_F32) {            // the fp32 kernels use 64 x 128 tiles and a smaller state
                    if (md != (dir ? P->pfwd[0].mode : P->pinv[0].mode)) continue;
                    const int nb32 = (P->Lp / SHT_TQ) * (R.ntp / 128);
                    P->skip_nb[dir][0] = nb32;
                    P->skip_p0[dir][0] = B.take<int>(nb32);
                    P->skip_state[dir][0] = reinterpret_cast<double*>(B.take<char>((size_t)nb32 * SHT_SKIP_STATE_BYTES_F32));
                    continue;
                }
                ThetaArgs t{};
                t.Lp = P->Lp; t.ntp = R.ntp; t.npass = np; t.nsm = P->nsm;
                t.tile = (P->opts & SHT_OPT_TILE64) ? 64 : (P->opts & SHT_OPT_TILE128) ? 128 : 0;
                const int nb = (P->Lp / SHT_TQ) * (R.ntp / theta_tile_rings(t)) * np;
                P->skip_nb[dir][md] = nb;
                P->skip_p0[dir][md] = B.take<int>(nb);
                P->skip_state[dir][md] = reinterpret_cast<double*>(B.take<char>((size_t)nb * SHT_SKIP_STATE_BYTES));
            }
    }
    if (P->precomp) {        // E[m - m_end][ntp][Lp] per pass: the O(L^3) memory of Sec. 4.3
        for (auto& ph : P->pinv) ph.p.pre = B.take<double>((size_t)(L - ph.p.m_end) * P->inv.ntp * Lp);
        for (auto& ph : P->pfwd) ph.p.pre = B.take<double>((size_t)(L - ph.p.m_end) * P->fwd.ntp * Lp);
    }
    if (P->batch > 1) {
        size_t oi = 0, of = 0;
        P->ob_off_inv.clear(); P->ob_off_fwd.clear();
        for (auto& ph : P->pinv) { P->ob_off_inv.push_back(oi); oi += (size_t)P->ncg * (L - ph.p.m_end) * P->inv.ntp * SHT_MMA_NCOL; }
        for (auto& ph : P->pfwd) { P->ob_off_fwd.push_back(of); of += (size_t)P->ncg_fwd * (L - ph.p.m_end) * Lp * SHT_MMA_NCOL; }
        P->Ob = B.take<double>(oi > of ? oi : of);
    }
    // scratch arrays (dimensions fixed by plan_dims)
    if (P->only_dir != 2) P->F = B.take<double2>(P->F_slab * P->nslab);
    P->polev = B.take<double2>(P->nslab);
    P->tmp = B.take<double>(2 * (size_t)Lp);
    P->unit_wq = B.take<double>(P->fwd.ntp);
    P->wq_map = B.take<double>(P->F_ld);
    P->wq_quad = B.take<double>(4 * (size_t)L);
    if (!P->helper) {
        if (P->sampling != SHT_HEALPIX) {
            P->Fa = B.take<double2>(P->Fa_slab * P->nslab);
            if (P->upsampled) P->X = B.take<double2>(P->X_slab * P->nslab);
        } else {
            P->it_map = B.take<double>(P->map_elems * (P->reality ? 1 : 2));
            P->it_coef = B.take<double>(2 * (size_t)L * P->M);
            if (P->io_f32) { P->it_f = B.take<double>(P->map_elems * (P->reality ? 1 : 2)); P->it_acc = B.take<double>(2 * (size_t)L * P->M); }
            P->hp_C = B.take<double2>((size_t)P->hp_ncap * P->hp_M);
            P->hp_BF = B.take<double2>((size_t)(P->hp_ncap / 2) * P->hp_M);
            P->hp_E = B.take<double2>((size_t)P->hp_neq * 4 * P->nside);
        }
        P->Z = B.take<double2>(P->Z_slab * P->nslab);
    }
    if (P->only_dir != 1) P->H = B.take<double2>(P->H_slab * P->nslab);
    if (P->reality && P->sampling != SHT_HEALPIX) P->cplx = B.take<double2>(P->map_elems * P->batch);
    if (P->kind == 1) P->fn = B.take<double2>((size_t)P->nslab * L * NB);
    if (P->io_f32) {
        const size_t ioe = (P->map_elems > (size_t)L * P->M ? P->map_elems : (size_t)L * P->M) * (P->kind == 1 ? P->nslab : 1);   // a map or a coefficient array
        P->io_a = B.take<double2>(ioe); P->io_b = B.take<double2>(ioe);
    }
    if (P->dtype == SHT_F32) {
        P->ab32 = B.take<float4>((size_t)L * Lp);
        P->st32_inv = B.take<float>((size_t)Lp * P->inv.ntp); P->k16_inv = B.take<uint16_t>((size_t)Lp * P->inv.ntp);
        P->st32_fwd = B.take<float>((size_t)Lp * P->fwd.ntp); P->k16_fwd = B.take<uint16_t>((size_t)Lp * P->fwd.ntp);
        P->lam32_inv = B.take<float>((size_t)(L + 1) * P->inv.ntp); P->lam32_fwd = B.take<float>((size_t)(L + 1) * P->fwd.ntp);
    }
    P->fft_work = B.take<char>(P->fft_work_bytes);
    // route every pass to its slab's output array
    for (auto& ph : P->pinv) ph.p.out = P->F ? P->F + P->F_slab * ph.p.slab + P->col0 : nullptr;   // regular ring th -> map ring col0 + th
    for (auto& ph : P->pfwd) ph.p.out = P->H ? P->H + P->H_slab * ph.p.slab : nullptr;
    if (P->batch > 1 && P->Ob) {
        for (size_t i = 0; i < P->pinv.size(); ++i) P->pinv[i].p.out = reinterpret_cast<double2*>(P->Ob + P->ob_off_inv[i]);
        for (size_t i = 0; i < P->pfwd.size(); ++i) P->pfwd[i].p.out = reinterpret_cast<double2*>(P->Ob + P->ob_off_fwd[i]);
    }
    if (!P->sub.empty()) {
        P->so3_dfwd = B.take<double>(L); P->so3_dinv = B.take<double>(L);
        P->adj_tmp = B.take<double2>((size_t)L * P->M);
    }
    // the helper plans of the adjoints live at the end of the same workspace
    for (sht_plan* Q : {P->adj_inv, P->adj_fwd})
        if (Q) { B.off = rup(B.off, 256); Q->work = base ? base + B.off : nullptr; B.off += Q->need_bytes; }
    for (sht_plan* Q : P->sub) { B.off = rup(B.off, 256); Q->work = base ? base + B.off : nullptr; B.off += Q->need_bytes; }
    P->need_bytes = rup(B.off, 256);
}

void add_passes(sht_plan* P, int slab, int n, bool real) {
    auto mk = [&](int nn, int sgn, int m_end, int mode, int mlo_key) {
        PassHost a{}; a.mode = mode;
        a.p.n = nn; a.p.sgn_out = sgn; a.p.m_end = m_end; a.p.slab = slab;
        (void)mlo_key;
        return a;
    };
    if (n == 0 && P->kind == 0) {
        PassHost a = mk(0, +1, 0, real ? 1 : 0, -1);
        P->pinv.push_back(a); P->pfwd.push_back(a);
        P->inv.start[0]; P->fwd.start[0];
    } else {
        // (SO(3) plans send n = 0 through the same two passes as the other orders, so that ONE launch serves all 2N-1 slabs: a
        //  separate +-m launch for the single n = 0 slab would occupy 8 blocks of the GPU for a whole recursion)
        int an = n < 0 ? -n : n;
        PassHost a = mk(n, +1, -an, 1, 2 * n), b = mk(-n, -1, 1 - an, 1, 2 * n + 1);
        // inverse on a ring set symmetric about the equator: ONE fold pass (+m at the ring, -m at the mirrored ring), as on the forward side
        const bool inv_fold = P->inv_fold && P->inv.symmetric;
        if (inv_fold) {
            PassHost c = mk(n, +1, -an, 0, 2 * n);
            c.p.fold = 1;
            P->pinv.push_back(c);
        } else { P->pinv.push_back(a); P->pinv.push_back(b); }
        // forward: the quadrature rings are symmetric about the equator, so ONE pass serves order +m from its own ring and order
        // -m from the mirrored ring (d^l_{-m,n}(pi - theta) = (-1)^{l-n} d^l_{m,n}(theta)): two orders per d-step
        if (P->fwd.symmetric) {
            PassHost c = mk(n, +1, -an, 0, 2 * n);
            c.p.fold = 1;
            P->pfwd.push_back(c);
            P->fwd.start[n]; P->fwd.mlo[2 * n];
        } else {        // (the MW rings, adjoint helper): no mirror ring to serve -m from: two passes, as on the inverse side
            P->pfwd.push_back(a); P->pfwd.push_back(b);
            P->fwd.start[n]; P->fwd.start[-n]; P->fwd.mlo[2 * n]; P->fwd.mlo[2 * n + 1];
        }
        if (inv_fold) { P->inv.start[n]; P->inv.mlo[2 * n]; }
        else { P->inv.start[n]; P->inv.start[-n]; P->inv.mlo[2 * n]; P->inv.mlo[2 * n + 1]; }
    }
}

sht_status make_fft_plans(sht_plan* P) {
    const int L = P->L, NB = P->NB;
    size_t ws = 0, w;
    if (P->sampling == SHT_HEALPIX) {
        const int ns = P->nside;
        P->hp_ncap = 2 * (ns - 1); P->hp_neq = 2 * ns + 1; P->hp_off_eq = 2LL * ns * (ns - 1);
        P->hp_M = 1;
        while (P->hp_M < 2 * 4 * (ns - 1) - 1) P->hp_M *= 2;
        if (P->hp_ncap > 0) {
            int nm[1] = {P->hp_M};
            CF(cufftCreate(&P->fft_hp_cap)); CF(cufftSetAutoAllocation(P->fft_hp_cap, 0));
            CF(cufftMakePlanMany(P->fft_hp_cap, 1, nm, nm, 1, P->hp_M, nm, 1, P->hp_M, CUFFT_Z2Z, P->hp_ncap, &w)); P->fft_elems[P->fft_hp_cap] = (double)P->hp_ncap * P->hp_M; ws = w > ws ? w : ws;
        }
        int ne[1] = {4 * ns};
        CF(cufftCreate(&P->fft_hp_eq)); CF(cufftSetAutoAllocation(P->fft_hp_eq, 0));
        CF(cufftMakePlanMany(P->fft_hp_eq, 1, ne, ne, 1, 4 * ns, ne, 1, 4 * ns, CUFFT_Z2Z, P->hp_neq, &w)); P->fft_elems[P->fft_hp_eq] = (double)P->hp_neq * 4 * ns; ws = w > ws ? w : ws;
        P->fft_work_bytes = ws + 256;
        P->have_fft = true;
        return SHT_OK;
    }
    // phi FFTs (Eq. 31 / 32): one ring per batch entry; F / Fa hold bin-major rows [bin][ring], the map is [ring][phi]
    const int nr = P->nrmap;
    int n1[1] = {NB};
    CF(cufftCreate(&P->fft_phi_inv)); CF(cufftSetAutoAllocation(P->fft_phi_inv, 0));
    { int inembed[1] = {NB}, onembed[1] = {NB};
      CF(cufftMakePlanMany(P->fft_phi_inv, 1, n1, inembed, P->F_ld, 1, onembed, 1, NB, CUFFT_Z2Z, nr, &w)); P->fft_elems[P->fft_phi_inv] = (double)nr * NB; ws = w > ws ? w : ws; }
    CF(cufftCreate(&P->fft_phi_fwd)); CF(cufftSetAutoAllocation(P->fft_phi_fwd, 0));
    { int inembed[1] = {NB}, onembed[1] = {NB};
      CF(cufftMakePlanMany(P->fft_phi_fwd, 1, n1, inembed, 1, NB, onembed, P->Ltp, 1, CUFFT_Z2Z, nr, &w)); P->fft_elems[P->fft_phi_fwd] = (double)nr * NB; ws = w > ws ? w : ws; }
    if (P->kind == 0 && P->batch == 1 && P->loop == 1 && !P->reality && !P->helper && L >= 1024) {
        for (int k : {8, 4, 2}) if (nr % k == 0) { P->nchunk = k; break; }
        if (P->nchunk) {
            int inembed[1] = {NB}, onembed[1] = {NB};
            CF(cufftCreate(&P->fft_phi_inv_c)); CF(cufftSetAutoAllocation(P->fft_phi_inv_c, 0));
            CF(cufftMakePlanMany(P->fft_phi_inv_c, 1, n1, inembed, P->F_ld, 1, onembed, 1, NB, CUFFT_Z2Z, nr / P->nchunk, &w)); P->fft_elems[P->fft_phi_inv_c] = (double)(nr / P->nchunk) * NB; ws = w > ws ? w : ws;
            CF(cufftCreate(&P->fft_phi_fwd_c)); CF(cufftSetAutoAllocation(P->fft_phi_fwd_c, 0));
            CF(cufftMakePlanMany(P->fft_phi_fwd_c, 1, n1, inembed, 1, NB, onembed, P->Ltp, 1, CUFFT_Z2Z, nr / P->nchunk, &w)); P->fft_elems[P->fft_phi_fwd_c] = (double)(nr / P->nchunk) * NB; ws = w > ws ? w : ws;
        }
    }
    if (P->upsampled) {
        // theta FFTs of the forward upsampling: length Tcirc on the extended samples, length 4L onto the quadrature rings
        int nt[1] = {P->Tcirc};
        CF(cufftCreate(&P->fft_th1)); CF(cufftSetAutoAllocation(P->fft_th1, 0));
        CF(cufftMakePlanMany(P->fft_th1, 1, nt, nt, 1, P->Tcirc, nt, 1, P->Tcirc, CUFFT_Z2Z, P->prow * P->nslab, &w)); P->fft_elems[P->fft_th1] = (double)P->Tcirc * P->prow * P->nslab; ws = w > ws ? w : ws;
        int n2[1] = {4 * L};
        CF(cufftCreate(&P->fft_th2)); CF(cufftSetAutoAllocation(P->fft_th2, 0));
        CF(cufftMakePlanMany(P->fft_th2, 1, n2, n2, 1, 4 * L, n2, 1, 4 * L, CUFFT_Z2Z, P->prow * P->nslab, &w)); P->fft_elems[P->fft_th2] = 4.0 * L * P->prow * P->nslab; ws = w > ws ? w : ws;
    }
    if (P->invsym) {
        int n4[1] = {2 * L};
        CF(cufftCreate(&P->fft_sym)); CF(cufftSetAutoAllocation(P->fft_sym, 0));
        CF(cufftMakePlanMany(P->fft_sym, 1, n4, n4, 1, 2 * L, n4, 1, 2 * L, CUFFT_Z2Z, P->prow, &w)); P->fft_elems[P->fft_sym] = 2.0 * L * P->prow; ws = w > ws ? w : ws;
    }
    if (P->kind == 1) {
        int n3[1] = {2 * P->N - 1};
        CF(cufftCreate(&P->fft_gamma)); CF(cufftSetAutoAllocation(P->fft_gamma, 0));
        int emb[1] = {2 * P->N - 1};
        CF(cufftMakePlanMany(P->fft_gamma, 1, n3, emb, L * NB, 1, emb, L * NB, 1, CUFFT_Z2Z, L * NB, &w)); P->fft_elems[P->fft_gamma] = (double)(2 * P->N - 1) * L * NB; ws = w > ws ? w : ws;
        CF(cufftCreate(&P->fft_alpha)); CF(cufftSetAutoAllocation(P->fft_alpha, 0));
        CF(cufftMakePlanMany(P->fft_alpha, 1, n1, n1, 1, NB, n1, 1, NB, CUFFT_Z2Z, L * P->nslab, &w)); P->fft_elems[P->fft_alpha] = (double)P->nslab * L * NB; ws = w > ws ? w : ws;
    }
    P->fft_work_bytes = ws + 256;
    P->have_fft = true;
    return SHT_OK;
}

// device of the calling thread and its SM count (tile and fold choices); without a device the defaults stand and the first
// CUDA / cuFFT call of plan creation reports the failure
void query_device(sht_plan* P) {
    int dev = 0, nsm = 0;
    if (cudaGetDevice(&dev) == cudaSuccess && cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess && nsm > 0) {
        P->device = dev; P->nsm = nsm;
    } else {
        (void)cudaGetLastError();
        P->device = 0; P->nsm = 148;
    }
}

// Eq. 27 start values are stored as a windowed double plus a one-byte window counter k, true value = stored * 2^(-SWIN k)
// (internal.h), which reaches down to 2^(TWIN - 255 SWIN) = 2^-122900.  |d^l_{l,n}(theta)| is smallest at l = L-1 on the ring nearest
// a pole; if it falls below that range the plan is refused (a start value is never silently dropped: the iterate grows back to
// O(1) at small m).  On MW this allows L up to ~9090.  log2 |d^l_{l,n}| = (1/2) log2 C(2l, l-n) + (l+n) log2 c2 + (l-n) log2 s2.
sht_status check_start_range(const sht_plan* P) {
    const ld floor2 = (ld)SHT_TWIN - 255.0L * (ld)SHT_SWIN;
    const int l = P->L - 1;
    for (const RingSet* R : {&P->inv, &P->fwd})
        for (int n : P->slab_n) {
            const int an = n < 0 ? -n : n;
            if (l < an) continue;
            const ld lb = (lgammal((ld)(2 * l + 1)) - lgammal((ld)(l + an + 1)) - lgammal((ld)(l - an + 1))) / (2.0L * logl(2.0L));
            for (int t : {0, R->nth - 1}) {
                if (t < 0 || t >= (int)R->c2.size()) continue;
                // both signs of n are recursed (mirror pass): take the smaller of the two magnitudes
                const ld a = (ld)(l + an) * log2l(R->c2[t]) + (ld)(l - an) * log2l(R->s2[t]);
                const ld b = (ld)(l - an) * log2l(R->c2[t]) + (ld)(l + an) * log2l(R->s2[t]);
                if (lb + (a < b ? a : b) < floor2 + 64) {
                    g_err = "band-limit too high for this ring set: Eq. 27 start values fall below the window-counter range 2^-122900";
                    return SHT_EUNSUPPORTED;
                }
            }
        }
    return SHT_OK;
}

sht_status plan_common(sht_plan* P) {
    const int L = P->L;
    P->Lp = (int)rup(L, 128);
    plan_dims(P);
    int nmax = 0;
    for (int n : P->slab_n) nmax = (n < 0 ? -n : n) > nmax ? (n < 0 ? -n : n) : nmax;
    P->kmin = -(nmax + 3);
    P->kstride = (int)rup((size_t)P->Lp + SHT_TQ + (size_t)(-P->kmin) + 2, 16);
    P->krows = P->Lp / SHT_TQ;
    P->mmin = -nmax - 1;           // one row below the lowest recursion step (dummy step of an odd final pair)
    P->sgstride = (int)rup((size_t)(L - P->mmin), 2);
    if (P->batch > 1) {            // one pass list serves every map of the batch
        add_passes(P, 0, P->slab_n[0], P->reality != 0);
        P->ncg = (P->batch * (P->pinv[0].mode == 0 ? 2 : 1) + 15) / 16;
        P->ncg_fwd = (P->batch * (P->pfwd[0].mode == 0 ? 2 : 1) + 15) / 16;
    } else
        for (int s = 0; s < P->nslab; ++s) add_passes(P, s, P->slab_n[s], P->reality != 0);
    if (P->only_dir == 1) { P->pfwd.clear(); P->fwd.start.clear(); P->fwd.mlo.clear(); }
    if (P->only_dir == 2) { P->pinv.clear(); P->inv.start.clear(); P->inv.mlo.clear(); }
    // d-step counts: rings * sum over l of the steps each pass runs
    for (int dir = 0; dir < 2; ++dir) {
        // algorithmic flop per d-step: 6 (recursion, as the paper states it) + 4 per order served and map
        double tot = 0, fl = 0; const RingSet& R = dir ? P->fwd : P->inv;
        for (auto& ph : (dir ? P->pfwd : P->pinv)) {
            int an = ph.p.n < 0 ? -ph.p.n : ph.p.n;
            double t = 0;
            for (int l = an; l < L; ++l) t += (double)(l - ph.p.m_end + 1);
            tot += t; fl += t * (6.0 + 4.0 * (ph.mode == 0 ? 2 : 1) * P->batch);
        }
        (dir ? P->dsteps_fwd : P->dsteps_inv) = tot * R.nth;
        (dir ? P->flops_fwd : P->flops_inv) = fl * R.nth;
    }
    if (!P->helper) CS(make_fft_plans(P));
    layout(P, nullptr);
    return SHT_OK;
}

// upload a host vector<double> through a staging copy (synchronous wrt the host buffer)
sht_status up(const std::vector<double>& h, double* d, cudaStream_t st) {
    CK(cudaMemcpyAsync(d, h.data(), h.size() * sizeof(double), cudaMemcpyHostToDevice, st));
    CK(cudaStreamSynchronize(st));
    return SHT_OK;
}

sht_status fill_ringset(sht_plan* P, RingSet& R, cudaStream_t st) {
    const int L = P->L, Lp = P->Lp;
    std::vector<double> csc(R.ntp, 1.0), tau(R.ntp, 0.0), sig(R.ntp, 1.0), c2h(R.ntp, 0.0), c2l(R.ntp, 0.0), s2h(R.ntp, 0.0), s2l(R.ntp, 0.0);
    for (int t = 0; t < R.nth; ++t) {
        ld c2 = R.c2[t], s2 = R.s2[t], st_ = 2 * c2 * s2;
        bool north = R.ct[t] >= 0;
        csc[t] = (double)(1 / st_);
        tau[t] = north ? (double)(s2 / c2) : (double)(-c2 / s2);
        sig[t] = north ? 1.0 : -1.0;
        c2h[t] = (double)c2; c2l[t] = (double)(c2 - (ld)c2h[t]);
        s2h[t] = (double)s2; s2l[t] = (double)(s2 - (ld)s2h[t]);
    }
    CS(up(csc, R.csc, st)); CS(up(tau, R.tau, st)); CS(up(sig, R.sig, st));
    CS(up(c2h, R.c2hi, st)); CS(up(c2l, R.c2lo, st)); CS(up(s2h, R.s2hi, st)); CS(up(s2l, R.s2lo, st));
    // start values per second index
    double* rtab = P->tmp;
    for (auto& kv : R.start) {
        int n = kv.first, an = n < 0 ? -n : n;
        std::vector<double> r(2 * (size_t)Lp, 0.0);
        for (int l = an + 1; l < L; ++l) {
            ld v = sqrtl((ld)(2 * l) * (ld)(2 * l - 1) / ((ld)(l + n) * (ld)(l - n)));
            r[l] = (double)v; r[Lp + l] = (double)(v - (ld)r[l]);
        }
        CS(up(r, rtab, st));
        CK(cudaMemsetAsync(kv.second.val, 0, sizeof(double) * (size_t)Lp * R.ntp, st));
        CK(cudaMemsetAsync(kv.second.k, 0, (size_t)Lp * R.ntp, st));
        CK(st_start_values(L, n, R.nth, R.ntp, R.c2hi, R.c2lo, R.s2hi, R.s2lo, rtab, rtab + Lp, kv.second.val, kv.second.k, P->d_flag, st));
        CK(cudaStreamSynchronize(st));
    }
    // peak split (R5): pass A serves m >= m_s = round(n cos theta), pass B serves m' >= 1 - m_s
    for (auto& kv : R.mlo) {
        int key = kv.first, n = (key - (key & 1)) / 2, passB = key & 1;
        std::vector<int> h(R.ntp, 1 << 30);
        for (int t = 0; t < R.nth; ++t) {
            // m_s(pi - theta) = -m_s(theta) exactly (the fold passes rely on it): evaluate on the northern ring of a mirror pair
            const int tm = R.nth - 1 - t;
            const bool mirrored = R.symmetric && tm < t;
            int ms = (int)llroundl((ld)n * R.ct[mirrored ? tm : t]);
            if (mirrored) ms = -ms;
            h[t] = passB ? 1 - ms : ms;
        }
        CK(cudaMemcpyAsync(kv.second, h.data(), sizeof(int) * R.ntp, cudaMemcpyHostToDevice, st));
        CK(cudaStreamSynchronize(st));
    }
    return SHT_OK;
}

sht_status upload_passes(sht_plan* P, cudaStream_t st) {
    for (int dir = 0; dir < 2; ++dir) {
        RingSet& R = dir ? P->fwd : P->inv;
        std::vector<ThetaPass> pm, p;
        for (auto& ph : (dir ? P->pfwd : P->pinv)) {
            ThetaPass t = ph.p;
            t.st_val = R.start[t.n].val; t.st_k = R.start[t.n].k;
            if (t.n != 0 || P->kind == 1) {      // (SO(3) plans route n = 0 through the general passes too)
                int n_slab = t.sgn_out > 0 ? t.n : -t.n;
                t.m_lo = R.mlo[2 * n_slab + (t.sgn_out > 0 ? 0 : 1)];
            } else t.m_lo = nullptr;
            ph.p = t;
            {   // zero the operand / lambda buffers once (their first row stays zero for good), then fill the lambda table
                const size_t rows = (size_t)(P->L - t.m_end + 1);
                const size_t in_doubles = pass_in_doubles(P, ph, dir != 0);
                CK(cudaMemsetAsync(const_cast<double*>(t.in), 0, in_doubles * sizeof(double), st));
                CK(cudaMemsetAsync(const_cast<double*>(t.lam), 0, rows * R.ntp * sizeof(double), st));
                CK(st_lamtab(t.n, R.nth, R.ntp, t.m_end, P->L - t.m_end, R.csc, R.tau, R.sig, const_cast<double*>(t.lam) + R.ntp, st));
            }
            (ph.mode == 0 && P->batch == 1 ? pm : p).push_back(t);
        }
        ThetaPass* dpm = dir ? P->d_fwd_pm : P->d_inv_pm; ThetaPass* dp = dir ? P->d_fwd_p : P->d_inv_p;
        if (!pm.empty()) CK(cudaMemcpyAsync(dpm, pm.data(), pm.size() * sizeof(ThetaPass), cudaMemcpyHostToDevice, st));
        if (!p.empty()) CK(cudaMemcpyAsync(dp, p.data(), p.size() * sizeof(ThetaPass), cudaMemcpyHostToDevice, st));
        CK(cudaStreamSynchronize(st));
        (dir ? P->n_fwd_pm : P->n_inv_pm) = (int)pm.size();
        (dir ? P->n_fwd_p : P->n_inv_p) = (int)p.size();
    }
    return SHT_OK;
}

// contiguous, balanced share of the kernel rings of one direction (every ring costs the same number of d-steps);
// shares differ by at most one ring: the first (nth mod n) shares get one more
void shard_range(const sht_plan* P, bool fwd, int* lo, int* hi) {
    const int nth = (fwd ? P->fwd : P->inv).nth, n = P->shard_n, i = P->shard_rank;
    const int q = nth / n, r = nth % n;
    *lo = i * q + (i < r ? i : r);
    *hi = *lo + q + (i < r ? 1 : 0);
}

ThetaArgs theta_args(const sht_plan* P, bool fwd, bool pm) {
    const RingSet& R = fwd ? P->fwd : P->inv;
    ThetaArgs a{};
    a.L = P->L; a.Lp = P->Lp; a.nth = R.nth; a.ntp = R.ntp; a.NB = P->NB;
    a.sg = P->sgtab; a.sgstride = P->sgstride; a.mmin = P->mmin; a.ctab = P->ctab;
    a.fold0 = fwd ? P->fold0 : P->fold0i;
    a.ldout = P->F_ld; a.nfull = R.nfull;
    shard_range(P, fwd, &a.th_lo, &a.th_hi);
    a.nsm = P->nsm; a.tile = (P->opts & SHT_OPT_TILE64) ? 64 : (P->opts & SHT_OPT_TILE128) ? 128 : 0;
    a.passes = fwd ? (pm ? P->d_fwd_pm : P->d_fwd_p) : (pm ? P->d_inv_pm : P->d_inv_p);
    a.npass = fwd ? (pm ? P->n_fwd_pm : P->n_fwd_p) : (pm ? P->n_inv_pm : P->n_inv_p);
    if (P->skip_ready) { a.skip_p0 = P->skip_p0[fwd ? 1 : 0][pm ? 0 : 1]; a.skip_state = P->skip_state[fwd ? 1 : 0][pm ? 0 : 1]; }
    return a;
}

// arguments of the fp32 kernels (theta_f32.cu) for one direction
F32Args f32_args(const sht_plan* P, bool fwd) {
    F32Args a{};
    const RingSet& R = fwd ? P->fwd : P->inv;
    const PassHost& ph = fwd ? P->pfwd[0] : P->pinv[0];
    a.L = P->L; a.Lp = P->Lp; a.nth = R.nth; a.ntp = R.ntp; a.NB = P->NB; a.ldout = fwd ? 0 : P->F_ld;
    a.fold0 = fwd ? P->fold0 : P->fold0i; a.nfull = R.nfull;
    a.ab = P->ab32; a.lam32 = fwd ? P->lam32_fwd : P->lam32_inv;
    a.st_val = fwd ? P->st32_fwd : P->st32_inv; a.st_k = fwd ? P->k16_fwd : P->k16_inv;
    a.in = reinterpret_cast<const float2*>(ph.p.in);
    a.out = fwd ? P->H : P->F + P->col0;             // (inverse: regular ring th -> map ring col0 + th)
    if (P->skip_ready) { a.skip_p0 = P->skip_p0[fwd ? 1 : 0][0]; a.skip_state = reinterpret_cast<float*>(P->skip_state[fwd ? 1 : 0][0]); }
    return a;
}
// Silent-head skip tables (internal.h ThetaArgs::skip_*), built once at sht_plan_set_workspace with the plan's own
// kernels: (1) PROBE -- one full recursion per launch on the zeroed operand tables; every block records the first pair of steps (at least 8
// steps below its ramp) in which any warp contributed; (2) the host turns that into p0 = the pairs a transform may skip: 8 steps of margin
// before the first contribution, a multiple of 8 pairs (the mbarrier phases of the operand ring and of the hand-off repeat every 8 pairs),
// and only if p0 lies below the ramp and its first window check; (3) DUMP -- the blocks with p0 > 0 run pairs [0, p0) and store their
// register state.  The tables depend on the ring set and the passes only, not on the data.
sht_status build_skip_tables(sht_plan* P, cudaStream_t st) {
    const int L = P->L, nlt = P->Lp / SHT_TQ;
    P->skip_pairs[0] = P->skip_pairs[1] = P->all_pairs[0] = P->all_pairs[1] = 0;
    if (P->dtype == SHT_F32) {
        // fp32 kernels (theta_f32.cu): every step projects every item there, so a skipped pair saves a whole pair.  Their recursion
        // coefficients are plan-time tables; the operand tables are still all zero at this point.
        for (int dir = 0; dir < 2; ++dir) {
            const int nb = P->skip_nb[dir][0];
            if (!nb) continue;
            F32Args a = f32_args(P, dir != 0);
            const int NC = (dir ? P->pfwd[0] : P->pinv[0]).mode == 0 ? 2 : 1, ntt = a.ntp / 128;
            a.skip_p0 = P->skip_p0[dir][0]; a.skip_state = reinterpret_cast<float*>(P->skip_state[dir][0]);
            CK(cudaMemsetAsync(a.skip_p0, 0, sizeof(int) * nb, st));
            a.skip_mode = 1;
            CK(launch_theta_f32(a, dir != 0, NC, st));
            std::vector<int> h(nb);
            CK(cudaMemcpyAsync(h.data(), a.skip_p0, sizeof(int) * nb, cudaMemcpyDeviceToHost, st));
            CK(cudaStreamSynchronize(st));
            for (int b = 0; b < nb; ++b) {
                const int lt = nlt - 1 - b / ntt, l0 = lt * SHT_TQ;
                const int mtop = l0 + SHT_TQ - 1 < L - 1 ? l0 + SHT_TQ - 1 : L - 1, npairs = (mtop + 2) / 2;
                int p0 = 0;
                if (h[b] > 0) {
                    p0 = (h[b] == (1 << 30) ? npairs : h[b]) - 4;
                    if (p0 < 4 || mtop - 2 * p0 >= l0 - 8) p0 = 0;
                }
                h[b] = p0;
                if (l0 < L) { P->all_pairs[dir] += npairs; P->skip_pairs[dir] += p0; }
            }
            CK(cudaMemcpyAsync(a.skip_p0, h.data(), sizeof(int) * nb, cudaMemcpyHostToDevice, st));
            a.skip_mode = 2;
            CK(launch_theta_f32(a, dir != 0, NC, st));
            CK(cudaStreamSynchronize(st));
        }
        P->skip_ready = true;
        return SHT_OK;
    }
    if (P->only_dir != 2 && P->H) {
        // the inverse kernels read their recursion coefficients g'_m(l), s_m from the operand rows that k_prep_inverse writes with every
        // transform: fill them once here, from all-zero harmonic coefficients (H serves as the zero array; the next transform zeroes it anyway)
        CK(cudaMemsetAsync(P->H, 0, sizeof(double2) * P->H_slab * P->nslab, st));
        CK(st_prep_inverse(L, P->Lp, 2, P->mmin, P->n_inv_pm, P->H, (size_t)L * P->M, P->d_cslab, P->scale_inv, P->ctab, P->sgtab, P->sgstride, P->d_inv_pm, st));
        CK(st_prep_inverse(L, P->Lp, 1, P->mmin, P->n_inv_p, P->H, (size_t)L * P->M, P->d_cslab, P->scale_inv, P->ctab, P->sgtab, P->sgstride, P->d_inv_p, st));
    }
    for (int dir = 0; dir < 2; ++dir) {
        if ((dir == 0 && P->only_dir == 2) || (dir == 1 && P->only_dir == 1)) continue;
        for (int md = 0; md < 2; ++md) {
            const int nb = P->skip_nb[dir][md];
            if (!nb) continue;
            ThetaArgs a = theta_args(P, dir != 0, md == 0);
            if (a.npass == 0) continue;
            const int rings = theta_tile_rings(a), ntt = a.ntp / rings;
            if (nlt * ntt * a.npass != nb) { g_err = "skip tables: block count mismatch"; return SHT_ECUDA; }
            a.skip_p0 = P->skip_p0[dir][md]; a.skip_state = P->skip_state[dir][md];
            CK(cudaMemsetAsync(a.skip_p0, 0, sizeof(int) * nb, st));
            a.skip_mode = 1;
            CK(dir ? launch_theta_forward(a, md, st) : launch_theta_inverse(a, md, st));
            std::vector<int> h(nb);
            CK(cudaMemcpyAsync(h.data(), a.skip_p0, sizeof(int) * nb, cudaMemcpyDeviceToHost, st));
            CK(cudaStreamSynchronize(st));
            std::vector<ThetaPass> passes(a.npass);
            CK(cudaMemcpy(passes.data(), a.passes, sizeof(ThetaPass) * a.npass, cudaMemcpyDeviceToHost));
            for (int b = 0; b < nb; ++b) {
                const int tile = b / a.npass, lt = nlt - 1 - tile / ntt, l0 = lt * SHT_TQ;
                const int mtop = l0 + SHT_TQ - 1 < L - 1 ? l0 + SHT_TQ - 1 : L - 1;
                const int npairs = (mtop - passes[b % a.npass].m_end + 2) / 2;
                int p0 = 0;
                if (h[b] > 0) {                              // (0: the block did not run)
                    const int first = h[b] == (1 << 30) ? npairs : h[b];
                    p0 = (first - 4) & ~7;
                    if (p0 < 8 || mtop - 2 * p0 >= l0 - 8) p0 = 0;
                }
                h[b] = p0;
                if (l0 < L) { P->all_pairs[dir] += npairs; P->skip_pairs[dir] += p0; }
            }
            CK(cudaMemcpyAsync(a.skip_p0, h.data(), sizeof(int) * nb, cudaMemcpyHostToDevice, st));
            a.skip_mode = 2;
            CK(dir ? launch_theta_forward(a, md, st) : launch_theta_inverse(a, md, st));
            CK(cudaStreamSynchronize(st));
        }
    }
    P->skip_ready = true;
    return SHT_OK;
}

MmaArgs mma_args(const sht_plan* P, bool fwd) {
    const RingSet& R = fwd ? P->fwd : P->inv;
    MmaArgs a{};
    a.L = P->L; a.Lp = P->Lp; a.nth = R.nth; a.ntp = R.ntp; a.ncg = fwd ? P->ncg_fwd : P->ncg; a.fold0 = fwd ? P->fold0 : 0;
    a.sg = P->sgtab; a.sgstride = P->sgstride; a.mmin = P->mmin;
    a.passes = fwd ? P->d_fwd_p : P->d_inv_p;
    a.npass = fwd ? P->n_fwd_p : P->n_inv_p;
    return a;
}

// cuFFT execution on `st` with byte accounting (an FFT pass reads and writes every element once: 32 B per complex element)
sht_status fft_exec(sht_plan* P, cufftHandle h, double2* in, double2* out, int dir, cudaStream_t st) {
    CF(cufftSetStream(h, st));
    CF(cufftExecZ2Z(h, in, out, dir));
    auto it = P->fft_elems.find(h);
    if (it != P->fft_elems.end()) count_bytes(32.0 * it->second);
    return SHT_OK;
}
sht_status zero_async(void* p, size_t bytes, cudaStream_t st) {
    CK(cudaMemsetAsync(p, 0, bytes, st));
    count_bytes((double)bytes);
    return SHT_OK;
}

// pole rings of the inverse ring set (the kernels skip them): theta = pi holds only the order m = -n (Eq. 29), theta = 0 only m = n
// (Eq. 28); F has been zeroed, so only those two entries are written.  Columns of F are in map-ring order.
sht_status inverse_poles(sht_plan* P, const double2* coef, cudaStream_t st) {
    const int L = P->L;
    const int nreg = P->inv.nfull ? P->inv.nfull : P->inv.nth;
    const size_t cs = (size_t)L * P->M;
    if (P->inv.pole && P->shard_rank == P->shard_n - 1)        // the south pole belongs to the last ring shard, the north pole to the first
        CK(st_pole_inverse(L, 0, P->NB, P->nslab, P->d_slab_n, P->d_cslab, coef, cs, P->scale_inv, P->F, P->F_slab, P->F_ld, P->col0 + nreg, st));
    if (P->inv.pole_n && P->shard_rank == 0)
        CK(st_pole_inverse(L, 1, P->NB, P->nslab, P->d_slab_n, P->d_cslab, coef, cs, P->scale_inv, P->F, P->F_slab, P->F_ld, 0, st));
    return SHT_OK;
}

// ---- the stages --------------------------------------------------------------------------------------------------
// coef: nslab slabs of [L][NB] in *slab order*.  Leaves F[slab][row][ring] complete (all rows, incl. the pole ring).
sht_status run_theta_inverse(sht_plan* P, const double2* coef, cudaStream_t st) {
    const int L = P->L;
    stage(P, CAT_STAGE, st);
    if (P->batch > 1) {
        // batched path: one recursion for all maps, contraction on FP64 tensor-core MMAs (theta_mma.cu).  All passes of a
        // plan have the same m_end up to 1, but their operand / result buffers are separate; the kernel takes the
        // column-group strides of the FIRST pass, so passes are launched one by one when their row counts differ.
        CS(zero_async(P->F, sizeof(double2) * P->F_slab * P->nslab, st));
        for (size_t i = 0; i < P->pinv.size(); ++i) {
            auto& ph = P->pinv[i];
            const int NC = ph.mode == 0 ? 2 : 1;
            const size_t rows = (size_t)(L - ph.p.m_end);
            CK(st_prep_inverse_batch(L, P->Lp, NC, P->batch, P->ncg, ph.p.n, ph.p.sgn_out, ph.p.m_end, P->mmin, coef, P->scale_inv,
                                     P->ctab, P->sgtab, P->sgstride, const_cast<double*>(ph.p.in), rows * P->Lp * SHT_MMA_ROW, st));
            CS(zero_async(ph.p.out, sizeof(double) * P->ncg * rows * P->inv.ntp * SHT_MMA_NCOL, st));
        }
        stage(P, CAT_HOT, st);
        for (size_t i = 0; i < P->pinv.size(); ++i) {
            MmaArgs a = mma_args(P, false);
            const size_t rows = (size_t)(L - P->pinv[i].p.m_end);
            a.passes += i; a.npass = 1;
            a.in_cg_stride = rows * P->Lp * SHT_MMA_ROW; a.out_cg_stride = rows * P->inv.ntp * SHT_MMA_NCOL;
            CK(launch_theta_mma(a, false, st));
        }
        stage(P, CAT_STAGE, st);
        for (size_t i = 0; i < P->pinv.size(); ++i) {
            auto& ph = P->pinv[i];
            const size_t rows = (size_t)(L - ph.p.m_end);
            CK(st_unpack_batch(L, P->Lp, P->inv.ntp, P->inv.nth, ph.mode == 0 ? 2 : 1, P->batch, P->ncg, ph.p.n, ph.p.sgn_out, ph.p.m_end,
                               P->mmin, 0, 0, P->ctab, reinterpret_cast<const double*>(ph.p.out), rows * P->inv.ntp * SHT_MMA_NCOL, P->F,
                               P->F_slab, P->inv.ntp, st));
        }
        CS(inverse_poles(P, coef, st));
        if (P->reality)
            for (int s = 0; s < P->nslab; ++s) CK(st_hermitian_rows(L, P->NB, P->F_ld, P->F_nrings, P->F + P->F_slab * s, st));
        return SHT_OK;
    }
    if (P->dtype == SHT_F32) {
        auto& ph = P->pinv[0];
        const int NC = ph.mode == 0 ? 2 : 1;
        CK(st_prep_inverse_f32(L, P->Lp, NC, coef, P->scale_inv, reinterpret_cast<float2*>(const_cast<double*>(ph.p.in)), st));
        CS(zero_async(P->F, sizeof(double2) * P->F_slab, st));
        stage(P, CAT_HOT, st);
        CK(launch_theta_f32(f32_args(P, false), false, NC, st));
        CS(inverse_poles(P, coef, st));
        stage(P, CAT_STAGE, st);
        if (P->reality) CK(st_hermitian_rows(L, P->NB, P->F_ld, P->F_nrings, P->F, st));
        return SHT_OK;
    }
    CK(st_prep_inverse(L, P->Lp, 2, P->mmin, P->n_inv_pm, coef, (size_t)L * P->M, P->d_cslab, P->scale_inv, P->ctab, P->sgtab, P->sgstride, P->d_inv_pm, st));
    CK(st_prep_inverse(L, P->Lp, 1, P->mmin, P->n_inv_p, coef, (size_t)L * P->M, P->d_cslab, P->scale_inv, P->ctab, P->sgtab, P->sgstride, P->d_inv_p, st));
    CS(zero_async(P->F, sizeof(double2) * P->F_slab * P->nslab, st));
    stage(P, CAT_HOT, st);
    if (P->precomp) {
        CK(launch_pre_inverse(theta_args(P, false, true), 0, L - P->mmin - 1, st));
        CK(launch_pre_inverse(theta_args(P, false, false), 1, L - P->mmin - 1, st));
    } else {
        CK(launch_theta_inverse(theta_args(P, false, true), 0, st));
        CK(launch_theta_inverse(theta_args(P, false, false), 1, st));
    }
    CS(inverse_poles(P, coef, st));
    stage(P, CAT_STAGE, st);
    if (P->reality)
        for (int s = 0; s < P->nslab; ++s) CK(st_hermitian_rows(L, P->NB, P->F_ld, P->F_nrings, P->F + P->F_slab * s, st));
    return SHT_OK;
}
// U: [slab][bin][ldu] samples of F_m on the forward ring set (weights not yet applied).  Leaves H complete.
// pair != 0: U is the paired output of mw_upsample (two orders per row, staging.cu u_get).
sht_status run_theta_forward(sht_plan* P, const double2* U, size_t U_slab, int ldu, cudaStream_t st, int pair = 0) {
    const int L = P->L;
    stage(P, CAT_STAGE, st);
    if (P->batch > 1) {
        CS(zero_async(P->H, sizeof(double2) * P->H_slab * P->nslab, st));
        for (size_t i = 0; i < P->pfwd.size(); ++i) {
            auto& ph = P->pfwd[i];
            const size_t rows = (size_t)(L - ph.p.m_end);
            if (P->fold0) {
                CK(st_weight_split_batch_fold0(L, P->NB, ldu, pair, U_slab, P->fwd.nth, P->fwd.ntp, P->fwd.nfull, ph.mode == 0 ? 2 : 1, P->batch,
                                               P->ncg_fwd, ph.p.m_end, P->fwd.wq, ph.p.lam, U, const_cast<double*>(ph.p.in),
                                               rows * P->fwd.ntp * SHT_MMA_ROWF, st));
                CS(zero_async(ph.p.out, sizeof(double) * P->ncg_fwd * rows * P->Lp * SHT_MMA_NCOL, st));
                continue;
            }
            CK(st_weight_split_batch(L, P->NB, ldu, pair, U_slab, P->fwd.nth, P->fwd.ntp, ph.mode == 0 ? 2 : 1, P->batch, P->ncg_fwd, P->slab_n[0],
                                     ph.p.sgn_out, ph.p.m_end, ph.p.fold, ph.p.m_lo, P->fwd.wq, ph.p.lam, U, const_cast<double*>(ph.p.in),
                                     rows * P->fwd.ntp * SHT_MMA_ROW, st));
            CS(zero_async(ph.p.out, sizeof(double) * P->ncg_fwd * rows * P->Lp * SHT_MMA_NCOL, st));
        }
        stage(P, CAT_HOT, st);
        for (size_t i = 0; i < P->pfwd.size(); ++i) {
            MmaArgs a = mma_args(P, true);
            const size_t rows = (size_t)(L - P->pfwd[i].p.m_end);
            a.passes += i; a.npass = 1;
            a.in_cg_stride = rows * P->fwd.ntp * (P->fold0 ? SHT_MMA_ROWF : SHT_MMA_ROW); a.out_cg_stride = rows * P->Lp * SHT_MMA_NCOL;
            CK(launch_theta_mma(a, true, st));
        }
        stage(P, CAT_STAGE, st);
        for (size_t i = 0; i < P->pfwd.size(); ++i) {
            auto& ph = P->pfwd[i];
            const size_t rows = (size_t)(L - ph.p.m_end);
            CK(st_unpack_batch(L, P->Lp, P->Lp, L, ph.mode == 0 ? 2 : 1, P->batch, P->ncg_fwd, ph.p.n, ph.p.sgn_out, ph.p.m_end, P->mmin, 1, ph.p.fold,
                               P->ctab, reinterpret_cast<const double*>(ph.p.out), rows * P->Lp * SHT_MMA_NCOL, P->H, P->H_slab, P->Lp, st));
        }
        return SHT_OK;
    }
    if (P->dtype == SHT_F32) {
        auto& ph = P->pfwd[0];
        const int NC = ph.mode == 0 ? 2 : 1;
        float2* W32 = reinterpret_cast<float2*>(const_cast<double*>(ph.p.in));
        if (P->fold0) CK(st_weight_split_f32_fold0(L, P->NB, ldu, pair, P->fwd.nth, P->fwd.ntp, P->fwd.nfull, NC, P->fwd.wq, U, W32, st));
        else CK(st_weight_split_f32(L, P->NB, ldu, pair, P->fwd.nth, P->fwd.ntp, NC, P->fwd.wq, U, W32, st));
        CS(zero_async(P->H, sizeof(double2) * P->H_slab, st));
        stage(P, CAT_HOT, st);
        CK(launch_theta_f32(f32_args(P, true), true, NC, st));
        return SHT_OK;
    }
    int slo, shi;
    shard_range(P, true, &slo, &shi);
    if (P->fold0) {         // n = 0 on the northern rings: E / O operand sets (one pass)
        for (auto& ph : P->pfwd) {
            const int NC = ph.mode == 0 ? 2 : 1;
            CK(st_weight_split_fold0(L, P->NB, ldu, pair, P->fwd.nth, P->fwd.ntp, P->fwd.nfull, NC, ph.p.m_end, P->fwd.wq, U + U_slab * ph.p.slab,
                                     reinterpret_cast<double2*>(const_cast<double*>(ph.p.in)) + (size_t)P->fwd.ntp * 2 * NC, slo, shi, st));
        }
    } else {
        CK(st_weight_split(L, P->NB, ldu, pair, P->fwd.nth, P->fwd.ntp, 2, P->mmin, P->n_fwd_pm, P->fwd.wq, U, U_slab, P->d_fwd_pm, slo, shi, st));
        CK(st_weight_split(L, P->NB, ldu, pair, P->fwd.nth, P->fwd.ntp, 1, P->mmin, P->n_fwd_p, P->fwd.wq, U, U_slab, P->d_fwd_p, slo, shi, st));
    }
    CS(zero_async(P->H, sizeof(double2) * P->H_slab * P->nslab, st));
    stage(P, CAT_HOT, st);
    if (P->precomp) {
        CK(launch_pre_forward(theta_args(P, true, true), 0, L - P->mmin - 1, st));
        CK(launch_pre_forward(theta_args(P, true, false), 1, L - P->mmin - 1, st));
    } else {
        CK(launch_theta_forward(theta_args(P, true, true), 0, st));
        CK(launch_theta_forward(theta_args(P, true, false), 1, st));
    }
    // pole rings of the ring set (only the adjoint helpers on the rings of an MW / MWSS map have any; unit weight): U points at
    // the first regular ring, the south pole follows the regular rings, the north pole precedes them
    const int nreg = P->fwd.nfull ? P->fwd.nfull : P->fwd.nth;
    for (int s = 0; s < P->nslab; ++s) {
        if (P->fwd.pole) CK(st_pole_forward(L, P->Lp, P->slab_n[s], 0, P->NB, ldu, nreg, 1.0, U + U_slab * s, P->H + P->H_slab * s, st));
        if (P->fwd.pole_n) CK(st_pole_forward(L, P->Lp, P->slab_n[s], 1, P->NB, ldu, -1, 1.0, U + U_slab * s, P->H + P->H_slab * s, st));
    }
    return SHT_OK;
}

sht_status check_ready(const sht_plan* P) {
    if (!P) return SHT_EINVAL;
    if (!P->ready) { g_err = "plan has no workspace (call sht_plan_set_workspace)"; return SHT_EWORKSPACE; }
    return SHT_OK;
}

// invsym: F[bin][F_ld] holds F_m on the L midpoint rings; replace it by F_m on the L MW rings (incl. the ring theta = pi).
// Scratch: Z (2L per row, FFT in place), X (2L-1 per row, inverse FFT in place).
sht_status resample_sym_to_mw(sht_plan* P, cudaStream_t st) {
    const int L = P->L, NB = P->NB;
    stage(P, CAT_STAGE, st);
    CK(st_sym_extend(L, P->slab_n[0], P->pair, P->F_ld, P->F, P->Z, st));
    stage(P, CAT_FFT, st);
    CS(fft_exec(P, P->fft_sym, P->Z, P->Z, CUFFT_FORWARD, st));
    stage(P, CAT_STAGE, st);
    CK(st_sym_rebin(L, P->prow, P->Z, P->X, st));
    stage(P, CAT_FFT, st);
    CS(fft_exec(P, P->fft_th1, P->X, P->X, CUFFT_INVERSE, st));
    stage(P, CAT_STAGE, st);
    if (P->pair) CK(st_sym_unpair(L, P->slab_n[0], P->F_ld, P->X, P->F, st));    // two orders per column: split them by their symmetry
    else CK(st_rows_head(NB, L, NB, P->F_ld, P->X, P->F, st));
    return SHT_OK;
}

// MW / MWSS: F_m on the rings of the map (Fa, [bin][Ltp]) -> U[bin][4L] on the rings theta'_u = (2u+1)pi/(4L) (in Z; u < 2L used)
sht_status mw_upsample(sht_plan* P, cudaStream_t st) {
    const int L = P->L, T2 = 4 * L, mwss = P->sampling == SHT_MWSS;
    stage(P, CAT_STAGE, st);
    // (with `pair` the rows are packed: slab stride prow rows, so that one batched FFT plan serves all slabs)
    const size_t xs = (size_t)P->prow * P->Tcirc, zs = (size_t)P->prow * T2;
    CK(st_mw_extend(L, P->nslab, P->d_slab_n, mwss, P->pair, P->Ltp, P->Tcirc, P->Fa, P->Fa_slab, P->X, xs, st));
    stage(P, CAT_FFT, st);
    CS(fft_exec(P, P->fft_th1, P->X, P->X, CUFFT_FORWARD, st));
    stage(P, CAT_STAGE, st);
    CK(st_mw_pad_phase(L, P->nslab, mwss, P->prow, P->Tcirc, T2, P->X, xs, P->Z, zs, st));
    stage(P, CAT_FFT, st);
    CS(fft_exec(P, P->fft_th2, P->Z, P->Z, CUFFT_INVERSE, st));
    return SHT_OK;
}

// HEALPix ring analysis: map -> U[bin(m)][ring] = e^{-i m phi0} DFT_ring[m mod nphi], in P->Z
sht_status healpix_analysis(sht_plan* P, const void* f, cudaStream_t st) {
    const int ns = P->nside, L = P->L, real = P->reality;
    const size_t nbelt = (size_t)P->hp_neq * 4 * ns;
    if (real) { stage(P, CAT_STAGE, st); CK(st_real_to_complex(nbelt, (const double*)f + P->hp_off_eq, P->hp_E, st)); }
    stage(P, CAT_FFT, st);
    CS(fft_exec(P, P->fft_hp_eq, real ? P->hp_E : const_cast<double2*>((const double2*)f + P->hp_off_eq), P->hp_E, CUFFT_FORWARD, st));
    if (P->hp_ncap > 0) {
        stage(P, CAT_STAGE, st);
        CK(st_hp_pack_fwd(ns, P->hp_M, real, f, P->hp_C, st));
        stage(P, CAT_FFT, st);
        CS(fft_exec(P, P->fft_hp_cap, P->hp_C, P->hp_C, CUFFT_FORWARD, st));
        stage(P, CAT_STAGE, st);
        CK(st_hp_mul(ns, P->hp_M, P->hp_BF, P->hp_C, st));
        stage(P, CAT_FFT, st);
        CS(fft_exec(P, P->fft_hp_cap, P->hp_C, P->hp_C, CUFFT_INVERSE, st));
    }
    stage(P, CAT_STAGE, st);
    CK(st_hp_unpack_fwd(ns, L, P->NB, real ? 0 : -(L - 1), P->fwd_ld, P->hp_M, P->hp_C, P->hp_E, P->Z, st));
    return SHT_OK;
}
// HEALPix ring synthesis: F[bin][ring] -> fold onto m mod nphi with the ring phase -> per-ring synthesis
sht_status healpix_synthesis(sht_plan* P, void* f, cudaStream_t st) {
    const int ns = P->nside, L = P->L, real = P->reality;
    const size_t nbelt = (size_t)P->hp_neq * 4 * ns;
    stage(P, CAT_STAGE, st);
    CK(st_hp_fold_inv(ns, L, P->NB, P->F_ld, P->hp_M, P->F, P->hp_C, P->hp_E, st));
    stage(P, CAT_FFT, st);
    CS(fft_exec(P, P->fft_hp_eq, P->hp_E, real ? P->hp_E : (double2*)f + P->hp_off_eq, CUFFT_INVERSE, st));
    if (real) { stage(P, CAT_STAGE, st); CK(st_hp_belt_real(nbelt, P->hp_E, (double*)f + P->hp_off_eq, st)); }
    if (P->hp_ncap > 0) {
        stage(P, CAT_FFT, st);
        CS(fft_exec(P, P->fft_hp_cap, P->hp_C, P->hp_C, CUFFT_FORWARD, st));
        stage(P, CAT_STAGE, st);
        CK(st_hp_mul(ns, P->hp_M, P->hp_BF, P->hp_C, st));
        stage(P, CAT_FFT, st);
        CS(fft_exec(P, P->fft_hp_cap, P->hp_C, P->hp_C, CUFFT_INVERSE, st));
        stage(P, CAT_STAGE, st);
        CK(st_hp_unpack_inv(ns, P->hp_M, real, P->hp_C, f, st));
    }
    stage(P, CAT_STAGE, st);
    return SHT_OK;
}

}  // namespace

void count_launch(int n) { g_launches += n; }
void count_bytes(double b) { g_bytes += b; }

extern "C" {

const char* sht_status_string(sht_status s) {
    switch (s) {
        case SHT_OK: return "SHT_OK";
        case SHT_EINVAL: return "SHT_EINVAL: invalid argument";
        case SHT_EUNSUPPORTED: return "SHT_EUNSUPPORTED: not implemented in this build";
        case SHT_EWORKSPACE: return "SHT_EWORKSPACE: workspace missing or too small";
        case SHT_ECUDA: return "SHT_ECUDA: CUDA runtime failure";
        case SHT_ECUFFT: return "SHT_ECUFFT: cuFFT failure";
    }
    return "unknown status";
}
const char* sht_last_error(void) { return g_err.c_str(); }
const char* sht_version(void) { return "b200sht 0.1 (sm_100a)"; }
long sht_launch_count(int reset) { long v = g_launches; if (reset) g_launches = 0; return v; }

sht_status sht_plan_s2(sht_plan** out, int L, int spin, int sampling, int nside, int reality, int dtype) {
    return sht_plan_s2_opts(out, L, spin, sampling, nside, reality, dtype, 1, 0u);
}
sht_status sht_plan_s2_batch(sht_plan** out, int L, int spin, int sampling, int nside, int reality, int dtype, int batch) {
    return sht_plan_s2_opts(out, L, spin, sampling, nside, reality, dtype, batch, 0u);
}
static sht_status make_s2_plan(sht_plan** out, int L, int spin, int sampling, int nside, int reality, int dtype, int batch, unsigned opts,
                               int only_dir, bool helper) {
    if (!out) return SHT_EINVAL;
    *out = nullptr;
    if (batch < 1 || batch > 1024) return SHT_EINVAL;
    const bool internal = helper && (sampling == SHT_INT_MWRINGS || sampling == SHT_INT_MWSSRINGS);
    if (L < 1 || L > 16384 || abs(spin) >= L || (reality && spin != 0) || ((sampling < SHT_MW || sampling > SHT_GL) && !internal)) return SHT_EINVAL;
    // batches run through the shared-recursion DMMA kernels on MW fp64 plans; on the other samplings and in fp32 the single-map path
    // runs map by map (same results, no shared recursion)
    int loop = 1;
    if (batch > 1 && (sampling != SHT_MW || dtype == SHT_F32) && !helper && !(opts & (SHT_OPT_PRECOMPUTE | SHT_OPT_ADJOINT))) { loop = batch; batch = 1; }
    if (batch > 1 && sampling != SHT_MW) return SHT_EUNSUPPORTED;
    if (sampling == SHT_HEALPIX && nside < 1) return SHT_EINVAL;
    if (dtype != SHT_F64 && dtype != SHT_F32) return SHT_EINVAL;
    if (opts & SHT_OPT_PRECOMPUTE) {
        // stored d-functions (Sec. 4.3): single-map fp64 plans; the tables hold every ring, so the folds are off
        if (batch != 1 || dtype != SHT_F64 || (opts & (SHT_OPT_FOLD_ON | SHT_OPT_INVSYM | SHT_OPT_ADJOINT))) return SHT_EUNSUPPORTED;
        opts |= SHT_OPT_NO_INVSYM;
        opts |= SHT_OPT_FOLD_OFF;
    }
    if ((opts & SHT_OPT_FOLD_ON) && (opts & SHT_OPT_FOLD_OFF)) return SHT_EINVAL;
    if ((opts & SHT_OPT_TILE64) && (opts & SHT_OPT_TILE128)) return SHT_EINVAL;
    if ((opts & SHT_OPT_INVSYM) && (opts & SHT_OPT_NO_INVSYM)) return SHT_EINVAL;
    if ((opts & SHT_OPT_GRAPH) && (opts & SHT_OPT_NO_GRAPH)) return SHT_EINVAL;
    // fp32 variant (BASELINE config 5): one map at a time, any sampling.  spin 0: the fp32 kernels; spin != 0: fp32 public arrays around the
    // fp64 kernels (the fp32 kernels recurse the second index n = 0 only)
    if (dtype == SHT_F32 && (batch != 1 || helper || (opts & SHT_OPT_ADJOINT))) return SHT_EUNSUPPORTED;
    const bool io_f32 = dtype == SHT_F32;
    if (io_f32 && spin != 0) dtype = SHT_F64;
    if (sampling == SHT_HEALPIX && nside > 8192) return SHT_EINVAL;
    sht_plan* P = new sht_plan();
    P->dtype = dtype; P->io_f32 = io_f32; P->opts = opts; P->helper = helper; P->only_dir = only_dir;
    P->precomp = (opts & SHT_OPT_PRECOMPUTE) != 0;
    P->kind = 0; P->L = L; P->spin = spin; P->sampling = sampling; P->nside = sampling == SHT_HEALPIX ? nside : 0; P->reality = reality ? 1 : 0;
    P->loop = loop;
    P->batch = batch; P->nslab = batch; P->slab_n.assign(batch, -spin);        // sY_lm ~ d^l_{m,-s}  (Eq. 9+10)
    query_device(P);
    // ring sets: `inv` = the rings of the map (inverse theta step), `fwd` = the rings the forward quadrature runs on
    switch (sampling) {
        case SHT_MW: rings_mw(P->inv, L); rings_mid(P->fwd, 2 * L); break;           // Eq. 37; upsampled to the 2L midpoint rings (R9)
        case SHT_MWSS: rings_mwss(P->inv, L); rings_mid(P->fwd, 2 * L); break;       // Eq. 39; same quadrature rings
        case SHT_DH: rings_mid(P->inv, 2 * L); rings_mid(P->fwd, 2 * L); break;      // Eq. 34: theta_t = (2t+1)pi/(4L) -- the midpoint rings themselves
        case SHT_GL: rings_gl(P->inv, L, nullptr); rings_gl(P->fwd, L, &P->gl_w); break;   // roots of P_L
        case SHT_INT_MWRINGS: rings_mw(P->inv, L); rings_mw(P->fwd, L); break;        // adjoint helper: the rings of an MW map
        case SHT_INT_MWSSRINGS: rings_mwss(P->inv, L); rings_mwss(P->fwd, L); break;  // adjoint helper: the rings of an MWSS map
        default: rings_healpix(P->inv, nside); rings_healpix(P->fwd, nside); break;
    }
    if (spin == 0) {
        // n = 0 fold (theta_kernels.cu FOLD): worth it once the northern half alone fills the GPU with >= 2 waves of 64 x 128 tiles
        // (L >= 2048 on MW on 148 SMs); SHT_OPT_FOLD_ON / SHT_OPT_FOLD_OFF override the choice
        const long tiles = (long)(rup(L, 128) / SHT_TQ) * (long)(rup((size_t)(P->fwd.nth + 1) / 2, 128) / 128) * (batch > 1 ? 4 : 1);
        bool on = tiles >= 2 * (long)P->nsm;
        if (opts & SHT_OPT_FOLD_ON) on = true;
        if (opts & SHT_OPT_FOLD_OFF) on = false;
        if (on && P->fwd.symmetric && only_dir != 1) { P->fold0 = 1; north_only(P->fwd); }
        // MW inverse: the MW rings (2t+1)pi/(2L-1) are not symmetric.  F_m is evaluated on the L midpoint rings (2j+1)pi/(2L) instead, with
        // the north-south fold (half the d-steps), and resampled to the MW rings with two FFT passes (resample_sym_to_mw; exact).
        // Default wherever the fold itself is worth it (L >= 2048 on 148 SMs): measured inverse totals 3.39 -> 3.13 ms at L = 2048,
        // 23.8 -> 21.0 ms at L = 4096, 171.3 -> 131.6 ms at L = 8192.  SHT_OPT_INVSYM / SHT_OPT_NO_INVSYM override.
        bool isym = on;
        if (opts & SHT_OPT_INVSYM) isym = true;
        if (opts & (SHT_OPT_NO_INVSYM | SHT_OPT_FOLD_OFF)) isym = false;
        isym = isym && sampling == SHT_MW && batch == 1 && !helper && !(opts & SHT_OPT_ADJOINT);      // (fp64 and fp32 plans)
        if (isym) { P->invsym = 1; P->fold0i = 1; rings_mid(P->inv, L); north_only(P->inv); }
        // the rings of the map are symmetric about the equator on every sampling but MW: fold the inverse too.  DH has 2L rings, so
        // its folded inverse does the work of an MW inverse; it is folded whatever the size.
        if ((on || sampling == SHT_DH) && !(opts & SHT_OPT_FOLD_OFF) && sampling != SHT_MW && batch == 1 && P->inv.symmetric && only_dir != 2) {
            P->fold0i = 1; north_only(P->inv);
        }
    }
    // MW / MWSS forward upsampling and the symmetric-ring resampling carry two orders per theta-circle column (staging.cu u_get); the
    // adjoint entry points run the transposed chain on single orders, so plans that offer them keep one order per column
    P->pair = (sampling == SHT_MW || sampling == SHT_MWSS) && !helper && !(opts & (SHT_OPT_ADJOINT | SHT_OPT_NO_PAIR));
    // silent-head skip of the fused kernels (build_skip_tables): single-map fp64 on-the-fly plans from L >= 1024
    P->skip = !helper && batch == 1 && !(opts & (SHT_OPT_PRECOMPUTE | SHT_OPT_NO_SKIP)) && L >= 1024;      // (fp64 and fp32 kernels)
    // launch-bound sizes replay a captured CUDA graph (run_transform below)
    P->use_graph = !helper && loop == 1 && ((L <= 512 && !(opts & SHT_OPT_NO_GRAPH)) || (opts & SHT_OPT_GRAPH));
    if (spin != 0 && batch == 1 && dtype == SHT_F64 && !(opts & SHT_OPT_NO_INVSYM)) {
        // spin != 0: d^l_{-m,n}(pi - theta) = (-1)^{l-n} d^l_{m,n}(theta) lets ONE pass of the inverse serve order +m at a ring and
        // order -m at its mirror ring -- 6 FP64 instructions per d-step instead of 2 x 4, half the recursions -- wherever the inverse rings are
        // symmetric about the equator: MWSS, DH, GL, HEALPix as they are; MW through the L midpoint rings + the exact FFT resampling of the spin-0
        // symmetric-ring inverse (SHT_OPT_INVSYM forces it; default from L >= 2048, where it wins -- measured spin 2 inverse totals: L = 2048
        // 4.90 -> 3.74 ms, L = 1024 0.854 -> 0.846 ms, L = 512 0.27 -> 0.39 ms; SHT_OPT_NO_INVSYM keeps two passes on the rings of the map.
        // HEALPix / DH / MWSS at L = 1024 spin 2: 1.47 -> 1.15, 1.45 -> 1.07, 0.78 -> 0.65 ms)
        P->inv_fold = true;
        const bool isym = sampling == SHT_MW && !helper && !(opts & SHT_OPT_ADJOINT) && (L >= 2048 || (opts & SHT_OPT_INVSYM));
        if (isym) { P->invsym = 1; rings_mid(P->inv, L); }
    }
    sht_status s = check_start_range(P);
    if (s == SHT_OK && (opts & SHT_OPT_ADJOINT) && !helper) {
        // adjoint entry points (Eq. 52 / 58): complex fp64 single-map plans
        if (batch != 1 || dtype != SHT_F64 || reality) { g_err = "SHT_OPT_ADJOINT needs a complex fp64 single-map plan"; s = SHT_EUNSUPPORTED; }
        else if (sampling == SHT_MW || sampling == SHT_MWSS) {
            const unsigned hopts = opts & ~(unsigned)(SHT_OPT_ADJOINT | SHT_OPT_INVSYM);
            s = make_s2_plan(&P->adj_inv, L, spin, sampling == SHT_MW ? SHT_INT_MWRINGS : SHT_INT_MWSSRINGS, 0, 0, dtype, 1, hopts, 2, true);
            if (s == SHT_OK) s = make_s2_plan(&P->adj_fwd, L, spin, SHT_DH, 0, 0, dtype, 1, hopts, 1, true);
        }
    }
    if (s == SHT_OK) s = plan_common(P);
    if (s != SHT_OK) { sht_plan_destroy(P); return s; }
    *out = P;
    return SHT_OK;
}
sht_status sht_plan_s2_opts(sht_plan** out, int L, int spin, int sampling, int nside, int reality, int dtype, int batch, unsigned opts) {
    return make_s2_plan(out, L, spin, sampling, nside, reality, dtype, batch, opts, 0, false);
}

sht_status sht_plan_so3(sht_plan** out, int L, int N, int dtype) { return sht_plan_so3_opts(out, L, N, dtype, 0u); }
sht_status sht_plan_so3_opts(sht_plan** out, int L, int N, int dtype, unsigned opts) {
    if (!out) return SHT_EINVAL;
    *out = nullptr;
    if (L < 1 || L > 16384 || N < 1 || N > L) return SHT_EINVAL;
    if (dtype != SHT_F64 && dtype != SHT_F32) return SHT_EINVAL;
    if (dtype == SHT_F32 && (opts & SHT_OPT_ADJOINT)) return SHT_EUNSUPPORTED;
    sht_plan* P = new sht_plan();
    P->io_f32 = dtype == SHT_F32;          // fp32 public arrays around the fp64 kernels (the orders n != 0 need them, see make_s2_plan)
    P->kind = 1; P->L = L; P->N = N; P->sampling = SHT_MW;
    P->nslab = 2 * N - 1;
    for (int b = 0; b < P->nslab; ++b) P->slab_n.push_back(b < N ? b : b - (2 * N - 1));   // gamma-FFT bin order
    query_device(P);
    rings_mw(P->inv, L); rings_mid(P->fwd, 2 * L);
    P->pair = 1;
    P->opts = opts & (SHT_OPT_ADJOINT | SHT_OPT_GRAPH | SHT_OPT_NO_GRAPH);
    P->use_graph = (L <= 512 && !(opts & SHT_OPT_NO_GRAPH)) || (opts & SHT_OPT_GRAPH);
    sht_status s = ((opts & SHT_OPT_GRAPH) && (opts & SHT_OPT_NO_GRAPH)) ? SHT_EINVAL : check_start_range(P);
    if (s == SHT_OK && (opts & SHT_OPT_ADJOINT)) {
        // Wigner adjoints: per order n the transposed spin transform with s = -n (Eq. 15-18), through one S^2 adjoint plan each
        for (int b = 0; b < P->nslab && s == SHT_OK; ++b) {
            sht_plan* Q = nullptr;
            s = make_s2_plan(&Q, L, -P->slab_n[b], SHT_MW, 0, 0, SHT_F64, 1, SHT_OPT_ADJOINT | SHT_OPT_NO_GRAPH, 0, false);
            if (Q) P->sub.push_back(Q);
        }
    }
    if (s == SHT_OK) s = plan_common(P);
    if (s != SHT_OK) { sht_plan_destroy(P); return s; }
    *out = P;
    return SHT_OK;
}
size_t sht_plan_workspace_bytes(const sht_plan* P) { return P ? P->need_bytes : 0; }
int sht_plan_batch(const sht_plan* P) { return P ? (P->loop > 1 ? P->loop : P->batch) : 0; }
int sht_plan_ntheta(const sht_plan* P, int forward) {
    if (!P) return 0;
    if (!forward) return P->F_nrings;
    const RingSet& R = P->fwd;
    return (R.nfull ? R.nfull : R.nth) + (R.pole ? 1 : 0);
}
double sht_plan_dsteps(const sht_plan* P, int forward) { return P ? (forward ? P->dsteps_fwd : P->dsteps_inv) : 0.0; }
double sht_plan_skip_fraction(const sht_plan* P, int forward) {
    if (!P || !P->skip_ready) return 0.0;
    const int d = forward ? 1 : 0;
    return P->all_pairs[d] > 0 ? P->skip_pairs[d] / P->all_pairs[d] : 0.0;
}
double sht_plan_flops(const sht_plan* P, int forward) { return P ? (forward ? P->flops_fwd : P->flops_inv) : 0.0; }

sht_status sht_plan_set_workspace(sht_plan* P, void* work, size_t work_bytes, sht_stream stream) {
    if (!P || !work) return SHT_EINVAL;
    if (work_bytes < P->need_bytes) { g_err = "workspace too small"; return SHT_EWORKSPACE; }
    if (reinterpret_cast<uintptr_t>(work) % 256 != 0) { g_err = "workspace must be 256-byte aligned (bulk-TMA operand rows)"; return SHT_EINVAL; }
    cudaStream_t st = (cudaStream_t)stream;
    for (auto& g : P->graphs) cudaGraphExecDestroy(g.exec);      // captured transforms point into the old workspace
    P->graphs.clear();
    P->work = work; P->work_bytes = work_bytes;
    layout(P, (char*)work);
    const int L = P->L, Lp = P->Lp;
    CK(cudaMemsetAsync(P->d_flag, 0, 64 * sizeof(int), st));
    {   // SO(3): internal slabs are in gamma-FFT bin order, the public coefficient array in n order (n + N - 1)
        std::vector<int> cs(P->nslab);
        for (int b = 0; b < P->nslab; ++b) cs[b] = P->kind == 1 ? P->slab_n[b] + P->N - 1 : b;
        CK(cudaMemcpyAsync(P->d_slab_n, P->slab_n.data(), sizeof(int) * P->nslab, cudaMemcpyHostToDevice, st));
        CK(cudaMemcpyAsync(P->d_cslab, cs.data(), sizeof(int) * P->nslab, cudaMemcpyHostToDevice, st));
        CK(cudaStreamSynchronize(st));
    }
    CK(st_rsq(2 * Lp + 64, P->rsq, st));
    CK(st_kexp(P->krows, P->kstride, P->kmin, P->kexp, st));
    CK(st_ctab(L, Lp, P->mmin, P->kstride, P->kmin, P->kexp, P->rsq, P->ctab, st));
    CK(st_sgtab(P->krows, P->sgstride, P->mmin, P->kstride, P->kmin, P->kexp, P->sgtab, st));
    std::vector<double> si(Lp, 0.0), sf(Lp, 0.0);
    for (int l = 0; l < L; ++l) {
        if (P->kind == 0) {
            double pref = ((P->spin & 1) ? -1.0 : 1.0) * (double)sqrtl((ld)(2 * l + 1) / (4 * PI_L));     // Eq. 30 / 33
            si[l] = pref; sf[l] = pref;
        } else {
            si[l] = (double)((ld)(2 * l + 1) / (8 * PI_L * PI_L));                                        // Eq. 13
            sf[l] = (double)(2 * PI_L / (ld)(2 * P->N - 1));                                              // q_Gamma
        }
    }
    CS(up(si, P->scale_inv, st)); CS(up(sf, P->scale_fwd, st));
    if (P->only_dir != 2) CS(fill_ringset(P, P->inv, st));
    if (P->only_dir != 1) CS(fill_ringset(P, P->fwd, st));
    { std::vector<double> ones(P->fwd.ntp, 1.0); CS(up(ones, P->unit_wq, st)); }
    CK(cudaMemsetAsync(P->wq_map, 0, sizeof(double) * P->F_ld, st));
    CK(cudaMemsetAsync(P->wq_quad, 0, sizeof(double) * 4 * (size_t)L, st));
    if (P->helper) {
        // helper plans of the adjoints: only tables and pass lists; the forward-type helper sums with unit weights (Eq. 56)
        if (P->only_dir != 1) CK(cudaMemcpyAsync(P->fwd.wq, P->unit_wq, sizeof(double) * P->fwd.ntp, cudaMemcpyDeviceToDevice, st));
        CS(upload_passes(P, st));
        CK(cudaStreamSynchronize(st));
        int hflag = 0;
        CK(cudaMemcpy(&hflag, P->d_flag, sizeof(int), cudaMemcpyDeviceToHost));
        if (hflag) { g_err = "Eq. 27 start values fall below the window-counter range on this ring set"; return SHT_EUNSUPPORTED; }
        P->ready = true;
        return SHT_OK;
    }
    CK(cudaMemsetAsync(P->fwd.wq, 0, sizeof(double) * P->fwd.ntp, st));
    if (P->upsampled) CK(st_mid_weights(L, 2 * L, (double)(2 * PI_L / (ld)P->NB), P->wq_quad, st));      // all 2L quadrature rings
    if (P->sampling == SHT_DH) CK(st_mid_weights(L, 2 * L, (double)(2 * PI_L / (ld)P->NB), P->wq_map, st));
    if (P->sampling == SHT_GL || P->sampling == SHT_HEALPIX) {
        std::vector<double> w(P->F_ld, 0.0);
        for (int t = 0; t < P->nrmap; ++t)
            w[t] = P->sampling == SHT_GL ? (double)(2 * PI_L / (ld)(2 * L - 1) * P->gl_w[t]) : (double)(4 * PI_L / (12.0L * (ld)P->nside * (ld)P->nside));
        CS(up(w, P->wq_map, st));
    }
    if (P->sampling == SHT_MW || P->sampling == SHT_MWSS || P->sampling == SHT_DH) {
        // forward quadrature weights q_u = q_Phi v_u on the 2L midpoint rings, q_Phi = 2 pi / (phi samples per ring).  MW / MWSS: Eq. 41-44
        // restated for that ring set (R9).  DH: the rings ARE the DH rings and v_u equals the DH weight of Eq. 36 (Fejer's first
        // rule: (2/L) sin(theta) sum_k sin((2k+1)theta)/(2k+1) = (1/L)(1 + 2 sum_j cos(2j theta)/(1-4j^2)); the oracle uses Eq. 36 as printed).
        CK(st_mid_weights(L, P->fwd.nth, (double)(2 * PI_L / (ld)P->NB), P->fwd.wq, st));
    } else if (P->sampling == SHT_GL) {
        // Gauss-Legendre weights 2/((1-x^2) P_L'(x)^2) times q_Phi = 2 pi/(2L-1)  (Eq. 45-46, reading R22)
        std::vector<double> w(P->fwd.ntp, 0.0);
        for (int t = 0; t < P->fwd.nth; ++t) w[t] = (double)(2 * PI_L / (ld)(2 * L - 1) * P->gl_w[t]);
        CS(up(w, P->fwd.wq, st));
    } else {
        // HEALPix: equal pixel weights 4 pi / Npix
        std::vector<double> w(P->fwd.ntp, 0.0);
        for (int t = 0; t < P->fwd.nth; ++t) w[t] = (double)(4 * PI_L / (12.0L * (ld)P->nside * (ld)P->nside));
        CS(up(w, P->fwd.wq, st));
    }
    CS(upload_passes(P, st));
    if (P->precomp) {
        for (int dir = 0; dir < 2; ++dir) {
            for (auto& ph : (dir ? P->pfwd : P->pinv))
                CK(cudaMemsetAsync(const_cast<double*>(ph.p.pre), 0, sizeof(double) * (size_t)(L - ph.p.m_end) * (dir ? P->fwd.ntp : P->inv.ntp) * Lp, st));
            for (int pm = 0; pm < 2; ++pm) {
                ThetaArgs a = theta_args(P, dir != 0, pm != 0);
                a.th_lo = 0; a.th_hi = a.nth;
                CK(launch_pre_fill(a, st));
            }
        }
    }
    for (sht_plan* Q : {P->adj_inv, P->adj_fwd})
        if (Q) CS(sht_plan_set_workspace(Q, Q->work, Q->need_bytes, stream));
    if (!P->sub.empty()) {
        // Wigner vs spin normalisation (n even): W_n = (q_Gamma / p(l)) F_s, (W^-1)_n = F_s^-1 ((2l+1)/(8 pi^2) / p(l)), p(l) = sqrt((2l+1)/(4 pi))
        std::vector<double> df(L), di(L);
        for (int l = 0; l < L; ++l) {
            const ld p = sqrtl((ld)(2 * l + 1) / (4 * PI_L));
            df[l] = (double)((2 * PI_L / (ld)(2 * P->N - 1)) / p);
            di[l] = (double)(((ld)(2 * l + 1) / (8 * PI_L * PI_L)) / p);
        }
        CS(up(df, P->so3_dfwd, st)); CS(up(di, P->so3_dinv, st));
        for (sht_plan* Q : P->sub) CS(sht_plan_set_workspace(Q, Q->work, Q->need_bytes, stream));
    }
    if (P->dtype == SHT_F32) {
        CK(st_ab32(L, Lp, P->ab32, st));
        CK(st_start32((size_t)Lp * P->inv.ntp, P->inv.start[0].val, P->inv.start[0].k, P->st32_inv, P->k16_inv, st));
        CK(st_start32((size_t)Lp * P->fwd.ntp, P->fwd.start[0].val, P->fwd.start[0].k, P->st32_fwd, P->k16_fwd, st));
        CK(st_f64_to_f32((size_t)(L + 1) * P->inv.ntp, P->pinv[0].p.lam, P->lam32_inv, st));
        CK(st_f64_to_f32((size_t)(L + 1) * P->fwd.ntp, P->pfwd[0].p.lam, P->lam32_fwd, st));
    }
    if (P->sampling != SHT_HEALPIX) {
        for (cufftHandle h : {P->fft_phi_inv, P->fft_phi_fwd, P->fft_th1, P->fft_th2, P->fft_phi_inv_c, P->fft_phi_fwd_c})
            if (h) CF(cufftSetWorkArea(h, P->fft_work));
        if (P->invsym) CF(cufftSetWorkArea(P->fft_sym, P->fft_work));
        if (P->kind == 1) { CF(cufftSetWorkArea(P->fft_gamma, P->fft_work)); CF(cufftSetWorkArea(P->fft_alpha, P->fft_work)); }
    } else {
        CF(cufftSetWorkArea(P->fft_hp_eq, P->fft_work));
        if (P->hp_ncap > 0) {
            // chirp spectra: FFT of the wrapped chirps of the nside-1 distinct cap lengths (run through the cap batch plan)
            CF(cufftSetWorkArea(P->fft_hp_cap, P->fft_work));
            CK(cudaMemsetAsync(P->hp_C, 0, sizeof(double2) * (size_t)P->hp_ncap * P->hp_M, st));
            CK(st_hp_chirp(P->nside, P->hp_M, P->hp_C, st));
            CS(fft_exec(P, P->fft_hp_cap, P->hp_C, P->hp_C, CUFFT_FORWARD, st));
            CK(cudaMemcpyAsync(P->hp_BF, P->hp_C, sizeof(double2) * (size_t)(P->hp_ncap / 2) * P->hp_M, cudaMemcpyDeviceToDevice, st));
        }
    }
    CK(cudaStreamSynchronize(st));
    int flag = 0;
    CK(cudaMemcpy(&flag, P->d_flag, sizeof(int), cudaMemcpyDeviceToHost));
    if (flag) { g_err = "Eq. 27 start values fall below the window-counter range on this ring set"; return SHT_EUNSUPPORTED; }
    P->skip_ready = false;
    if (P->skip) CS(build_skip_tables(P, st));
    P->ready = true;
    return SHT_OK;
}

sht_status sht_plan_destroy(sht_plan* P) {
    if (!P) return SHT_OK;
    if (P->have_fft || P->fft_phi_inv) {
        for (cufftHandle h : {P->fft_phi_inv, P->fft_phi_fwd, P->fft_th1, P->fft_th2, P->fft_gamma, P->fft_alpha, P->fft_hp_cap, P->fft_hp_eq, P->fft_sym,
                              P->fft_phi_inv_c, P->fft_phi_fwd_c})
            if (h) cufftDestroy(h);
    }
    for (auto e : P->ev) cudaEventDestroy(e);
    for (auto& g : P->graphs) cudaGraphExecDestroy(g.exec);
    if (P->cap_stream) cudaStreamDestroy(P->cap_stream);
    if (P->copy_stream) cudaStreamDestroy(P->copy_stream);
    for (auto e : P->ev_copy) if (e) cudaEventDestroy(e);
    if (P->ev_begin) cudaEventDestroy(P->ev_begin);
    sht_plan_destroy(P->adj_inv); sht_plan_destroy(P->adj_fwd);
    for (sht_plan* Q : P->sub) sht_plan_destroy(Q);
    delete P;
    return SHT_OK;
}

sht_status sht_plan_enable_timing(sht_plan* P, int on) {
    if (!P) return SHT_EINVAL;
    if (on && P->ev.empty()) {
        P->ev.resize(96); P->ev_cat.assign(96, 0);
        for (auto& e : P->ev) CK(cudaEventCreate(&e));
    }
    P->timing = on != 0;
    return SHT_OK;
}
sht_status sht_plan_timings(sht_plan* P, float ms[4]) {
    if (!P || !ms) return SHT_EINVAL;
    ms[0] = ms[1] = ms[2] = ms[3] = 0.f;
    if (P->ev_n < 2) return SHT_OK;
    CK(cudaEventSynchronize(P->ev[P->ev_n - 1]));
    for (int i = 0; i + 1 < P->ev_n; ++i) {
        float t = 0.f;
        CK(cudaEventElapsedTime(&t, P->ev[i], P->ev[i + 1]));
        ms[P->ev_cat[i]] += t; ms[3] += t;
    }
    return SHT_OK;
}

sht_status sht_plan_set_shard(sht_plan* P, int rank, int nranks) {
    if (!P || nranks < 1 || rank < 0 || rank >= nranks) return SHT_EINVAL;
    bool mirror_writes = false;      // an inverse fold pass writes the -m orders of the MIRRORED rings: not confined to a ring share
    for (auto& ph : P->pinv) mirror_writes = mirror_writes || ph.p.fold;
    if (nranks > 1 && (P->batch > 1 || P->loop > 1 || P->dtype != SHT_F64 || P->io_f32 || P->invsym || mirror_writes || (P->opts & SHT_OPT_ADJOINT))) {   // (precompute plans shard too)
        g_err = "ring shards need a single-map fp64 plan created with SHT_OPT_NO_INVSYM and without SHT_OPT_ADJOINT";
        return SHT_EUNSUPPORTED;
    }
    P->shard_rank = rank; P->shard_n = nranks;
    for (auto& g : P->graphs) cudaGraphExecDestroy(g.exec);      // captured transforms carry the old share
    P->graphs.clear();
    return SHT_OK;
}
sht_status sht_plan_shard_range(const sht_plan* P, int forward, int* first, int* count) {
    if (!P || !first || !count) return SHT_EINVAL;
    int lo, hi;
    shard_range(P, forward != 0, &lo, &hi);
    *first = lo; *count = hi - lo;
    return SHT_OK;
}
sht_status sht_plan_stage_bytes(const sht_plan* P, double bytes[3]) {
    if (!P || !bytes) return SHT_EINVAL;
    for (int i = 0; i < 3; ++i) bytes[i] = P->sec_bytes[i];
    return SHT_OK;
}

// ---- S^2 ----------------------------------------------------------------------------------------------------------
sht_status s2_theta_inverse_plan(sht_plan* P, const void* flm, void* Fm, sht_stream stream) {
    CS(check_ready(P));
    if (!flm || !Fm || P->kind != 0) return SHT_EINVAL;
    if (P->batch > 1 || P->loop > 1 || P->dtype != SHT_F64 || P->io_f32) return SHT_EUNSUPPORTED;
    cudaStream_t st = (cudaStream_t)stream;
    begin_transform(P);
    CS(run_theta_inverse(P, (const double2*)flm, st));
    if (P->invsym) CS(resample_sym_to_mw(P, st));
    int nt = sht_plan_ntheta(P, 0);
    CK(st_rows_reorder(P->L, P->NB, nt, P->F_ld, nt, 1, P->F, (double2*)Fm, st));
    stage(P, CAT_STAGE, st);
    return SHT_OK;
}
sht_status s2_theta_forward_plan(sht_plan* P, const void* Wm, void* flm, sht_stream stream) {
    CS(check_ready(P));
    if (!Wm || !flm || P->kind != 0) return SHT_EINVAL;
    if (P->batch > 1 || P->loop > 1 || P->dtype != SHT_F64 || P->io_f32) return SHT_EUNSUPPORTED;
    cudaStream_t st = (cudaStream_t)stream;
    begin_transform(P);
    // this entry point takes rows that already carry the quadrature weight, so the split runs with unit weights
    int nt = sht_plan_ntheta(P, 1), T2 = P->fwd_ld;
    CK(st_rows_reorder(P->L, P->NB, nt, nt, T2, 0, (const double2*)Wm, P->Z, st));
    double* saved = P->fwd.wq;
    P->fwd.wq = P->unit_wq;
    sht_status s = run_theta_forward(P, P->Z, P->Z_slab, T2, st);
    P->fwd.wq = saved;
    if (s == SHT_OK) {
        stage(P, CAT_STAGE, st);
        cudaError_t e = st_finalize_forward(P->L, P->Lp, 1, P->d_slab_n, P->d_cslab, P->reality, P->scale_fwd, P->H, P->H_slab, (double2*)flm, 0, st);
        if (e != cudaSuccess) s = SHT_ECUDA;
        stage(P, CAT_STAGE, st);
    }
    return s;
}

static sht_status s2_inverse_body(sht_plan* P, const void* flm, void* f, sht_stream stream) {
    cudaStream_t st = (cudaStream_t)stream;
    const int L = P->L;
    const size_t ncoef = (size_t)L * P->M, nmap = P->map_elems;
    if (P->io_f32 && !P->f32_inner) {      // fp32 public arrays: fp64 copies around the core (staging and FFTs are fp64)
        CK(st_f32_to_f64(2 * ncoef, (const float*)flm, (double*)P->io_a, st));
        P->f32_inner = true;
        sht_status s = s2_inverse_body(P, P->io_a, P->io_b, stream);
        P->f32_inner = false;
        if (s != SHT_OK) return s;
        CK(st_f64_to_f32(P->reality ? nmap : 2 * nmap, (const double*)P->io_b, (float*)f, st));
        stage(P, CAT_STAGE, st);
        return SHT_OK;
    }
    begin_transform(P);
    CS(run_theta_inverse(P, (const double2*)flm, st));
    if (P->sampling == SHT_HEALPIX) return healpix_synthesis(P, f, st);
    if (P->invsym) CS(resample_sym_to_mw(P, st));
    if (P->skip_phi) return SHT_OK;                  // (host-buffer call: the ring synthesis runs chunk by chunk, overlapped with the copies out)
    stage(P, CAT_FFT, st);
    double2* outc = P->reality ? P->cplx : (double2*)f;
    for (int b = 0; b < P->batch; ++b)
        CS(fft_exec(P, P->fft_phi_inv, P->F + P->F_slab * b, outc + nmap * b, CUFFT_INVERSE, st));   // Eq. 32
    if (P->reality) { stage(P, CAT_STAGE, st); CK(st_complex_to_real(nmap * P->batch, P->cplx, (double*)f, st)); }
    stage(P, CAT_STAGE, st);
    return SHT_OK;
}
static sht_status s2_forward_body(sht_plan* P, const void* f, void* flm, sht_stream stream) {
    cudaStream_t st = (cudaStream_t)stream;
    const int L = P->L;
    const size_t ncoef = (size_t)L * P->M, nmap = P->map_elems;
    if (P->io_f32 && !P->f32_inner) {
        CK(st_f32_to_f64(P->reality ? nmap : 2 * nmap, (const float*)f, (double*)P->io_a, st));
        P->f32_inner = true;
        sht_status s = s2_forward_body(P, P->io_a, P->io_b, stream);
        P->f32_inner = false;
        if (s != SHT_OK) return s;
        CK(st_f64_to_f32(2 * ncoef, (const double*)P->io_b, (float*)flm, st));
        stage(P, CAT_STAGE, st);
        return SHT_OK;
    }
    begin_transform(P);
    if (P->sampling == SHT_HEALPIX) {
        CS(healpix_analysis(P, f, st));
        CS(run_theta_forward(P, P->Z, P->Z_slab, P->fwd_ld, st));
        stage(P, CAT_STAGE, st);
        CK(st_finalize_forward(L, P->Lp, 1, P->d_slab_n, P->d_cslab, P->reality, P->scale_fwd, P->H, P->H_slab, (double2*)flm, 0, st));
        stage(P, CAT_STAGE, st);
        return SHT_OK;
    }
    const double2* fin = (const double2*)f;
    if (P->reality) { stage(P, CAT_STAGE, st); CK(st_real_to_complex(nmap * P->batch, (const double*)f, P->cplx, st)); fin = P->cplx; }
    stage(P, CAT_FFT, st);
    for (int b = 0; b < P->batch && !P->skip_phi; ++b)                                 // Eq. 31 (weight folded into q_u)
        CS(fft_exec(P, P->fft_phi_fwd, const_cast<double2*>(fin) + nmap * b, P->Fa + P->Fa_slab * b, CUFFT_FORWARD, st));
    if (P->upsampled) {         // MW / MWSS: extension to the theta circle + upsampling to the quadrature rings
        CS(mw_upsample(P, st));
        CS(run_theta_forward(P, P->Z, (size_t)P->prow * P->fwd_ld, P->fwd_ld, st, P->pair));
    } else                      // DH / GL: explicit quadrature on the rings of the map (Eq. 36 / 46)
        CS(run_theta_forward(P, P->Fa, P->Fa_slab, P->Ltp, st));
    stage(P, CAT_STAGE, st);
    CK(st_finalize_forward(L, P->Lp, P->batch, P->d_slab_n, P->d_cslab, P->reality, P->scale_fwd, P->H, P->H_slab, (double2*)flm, ncoef, st));
    stage(P, CAT_STAGE, st);
    return SHT_OK;
}

// HEALPix forward transform with iterative refinement (the scheme has no sampling theorem, "iterations are usually
// performed"): flm_0 = F f;  flm_{k+1} = flm_k + F (f - F^-1 flm_k) -- Jacobi iterations on the residual map, every F / F^-1 the fused
// transforms above (reading R24 of DESIGN.md).  niter = 0 is s2_forward_plan.
sht_status s2_forward_iter_plan(sht_plan* P, const void* f, void* flm, int niter, sht_stream stream) {
    CS(check_ready(P));
    if (!flm || !f || P->kind != 0 || niter < 0) return SHT_EINVAL;
    if (P->sampling != SHT_HEALPIX) { g_err = "iterative refinement is a HEALPix feature: the other samplings are exact"; return SHT_EUNSUPPORTED; }
    if (P->loop > 1) { g_err = "iterative refinement is a single-map call"; return SHT_EUNSUPPORTED; }
    cudaStream_t st = (cudaStream_t)stream;
    const size_t nm = P->map_elems * (P->reality ? 1 : 2), nc = 2 * (size_t)P->L * P->M;
    if (P->io_f32) {
        // fp32 public arrays: the map, the running coefficients and the residual are kept in fp64 between the transforms (whose hot kernels
        // compute in fp32 for spin 0), so the iteration converges to what the transforms resolve, not to the rounding of the arrays
        CK(st_f32_to_f64(nm, (const float*)f, P->it_f, st));
        P->f32_inner = true;
        sht_status s = s2_forward_body(P, P->it_f, P->it_acc, stream);
        for (int it = 0; it < niter && s == SHT_OK; ++it) {
            s = s2_inverse_body(P, P->it_acc, P->it_map, stream);
            if (s == SHT_OK) s = st_vec_sub(nm, P->it_f, P->it_map, P->it_map, st) == cudaSuccess ? SHT_OK : SHT_ECUDA;
            if (s == SHT_OK) s = s2_forward_body(P, P->it_map, P->it_coef, stream);
            if (s == SHT_OK) s = st_vec_add(nc, P->it_coef, P->it_acc, st) == cudaSuccess ? SHT_OK : SHT_ECUDA;
        }
        P->f32_inner = false;
        if (s != SHT_OK) return s;
        CK(st_f64_to_f32(nc, P->it_acc, (float*)flm, st));
        return SHT_OK;
    }
    CS(s2_forward_plan(P, f, flm, stream));
    for (int it = 0; it < niter; ++it) {
        CS(s2_inverse_plan(P, flm, P->it_map, stream));
        CK(st_vec_sub(nm, (const double*)f, P->it_map, P->it_map, st));
        CS(s2_forward_plan(P, P->it_map, P->it_coef, stream));
        CK(st_vec_add(nc, P->it_coef, (double*)flm, st));
    }
    return SHT_OK;
}

// ---- adjoints (Sec. 5.3-5.4) -----------------------------------------------------------------------------------
namespace {
sht_status check_adjoint(const sht_plan* P) {
    if (!(P->opts & SHT_OPT_ADJOINT)) { g_err = "plan was not created with SHT_OPT_ADJOINT"; return SHT_EUNSUPPORTED; }
    return SHT_OK;
}
// forward-type kernel with unit weights on the rings of the map: U = F_m on those rings ([bin][ld], columns in map-ring order)
sht_status adjoint_analysis(sht_plan* P, const double2* U, size_t U_slab, int ldu, double2* flm, cudaStream_t st) {
    if (P->adj_inv) {           // MW / MWSS: helper plan on the rings of the map; U points at its first regular ring
        sht_plan* Q = P->adj_inv;
        CS(run_theta_forward(Q, U + P->col0, U_slab, ldu, st));
        CK(st_finalize_forward(P->L, Q->Lp, 1, Q->d_slab_n, Q->d_cslab, 0, Q->scale_fwd, Q->H, Q->H_slab, flm, 0, st));
        return SHT_OK;
    }
    double* saved = P->fwd.wq;
    P->fwd.wq = P->unit_wq;
    sht_status s = run_theta_forward(P, U, U_slab, ldu, st);
    P->fwd.wq = saved;
    CS(s);
    CK(st_finalize_forward(P->L, P->Lp, 1, P->d_slab_n, P->d_cslab, 0, P->scale_fwd, P->H, P->H_slab, flm, 0, st));
    return SHT_OK;
}
// inverse-type kernel on the quadrature rings: returns the array [bins][ld] holding F_m on ALL quadrature rings (unweighted)
sht_status adjoint_synthesis(sht_plan* P, const double2* flm, const double2** Fq, int* NBq, int* ldq, cudaStream_t st) {
    sht_plan* Q = P->adj_fwd ? P->adj_fwd : P;      // MW / MWSS: helper plan on the 2L midpoint rings
    CS(run_theta_inverse(Q, flm, st));
    *Fq = Q->F; *NBq = Q->NB; *ldq = Q->F_ld;
    return SHT_OK;
}
}  // namespace

sht_status s2_inverse_adjoint_plan(sht_plan* P, const void* f, void* flm, sht_stream stream) {
    CS(check_ready(P));
    if (!flm || !f || P->kind != 0) return SHT_EINVAL;
    CS(check_adjoint(P));
    cudaStream_t st = (cudaStream_t)stream;
    begin_transform(P);
    if (P->sampling == SHT_HEALPIX) {
        CS(healpix_analysis(P, f, st));                                          // ring DFTs with the ring phases: conj. transpose of Eq. 32
        return adjoint_analysis(P, P->Z, P->Z_slab, P->fwd_ld, (double2*)flm, st);
    }
    CS(fft_exec(P, P->fft_phi_fwd, (double2*)const_cast<void*>(f), P->Fa, CUFFT_FORWARD, st));
    return adjoint_analysis(P, P->Fa, P->Fa_slab, P->Ltp, (double2*)flm, st);
}
sht_status s2_theta_inverse_adjoint_plan(sht_plan* P, const void* Fm, void* flm, sht_stream stream) {
    CS(check_ready(P));
    if (!flm || !Fm || P->kind != 0) return SHT_EINVAL;
    CS(check_adjoint(P));
    cudaStream_t st = (cudaStream_t)stream;
    begin_transform(P);
    const int nt = sht_plan_ntheta(P, 0);
    double2* U = P->sampling == SHT_HEALPIX ? P->Z : P->Fa;
    const int ldu = P->sampling == SHT_HEALPIX ? P->fwd_ld : P->Ltp;
    CK(st_rows_reorder(P->L, P->NB, nt, nt, ldu, 0, (const double2*)Fm, U, st));
    return adjoint_analysis(P, U, P->sampling == SHT_HEALPIX ? P->Z_slab : P->Fa_slab, ldu, (double2*)flm, st);
}
sht_status s2_theta_forward_adjoint_plan(sht_plan* P, const void* flm, void* Wm, sht_stream stream) {
    CS(check_ready(P));
    if (!flm || !Wm || P->kind != 0) return SHT_EINVAL;
    CS(check_adjoint(P));
    cudaStream_t st = (cudaStream_t)stream;
    begin_transform(P);
    const double2* Fq; int NBq, ldq;
    CS(adjoint_synthesis(P, (const double2*)flm, &Fq, &NBq, &ldq, st));
    const int nq = sht_plan_ntheta(P, 1);
    CK(st_rows_reorder(P->L, NBq, nq, ldq, nq, 1, Fq, (double2*)Wm, st));
    return SHT_OK;
}
sht_status s2_forward_adjoint_plan(sht_plan* P, const void* flm, void* f, sht_stream stream) {
    CS(check_ready(P));
    if (!flm || !f || P->kind != 0) return SHT_EINVAL;
    CS(check_adjoint(P));
    cudaStream_t st = (cudaStream_t)stream;
    const int L = P->L;
    begin_transform(P);
    const double2* Fq; int NBq, ldq;
    CS(adjoint_synthesis(P, (const double2*)flm, &Fq, &NBq, &ldq, st));
    if (!P->upsampled) {
        // direct quadrature (DH, GL, HEALPix): F = Y^H Q, so F^H = Q Y -- Eq. 52 literally: weight the rings, then the ring synthesis
        CK(st_scale_cols(P->NB, P->nrmap, P->F_ld, P->wq_map, P->F, st));
        if (P->sampling == SHT_HEALPIX) return healpix_synthesis(P, f, st);
        return fft_exec(P, P->fft_phi_inv, P->F, (double2*)f, CUFFT_INVERSE, st);
    }
    // MW / MWSS: conjugate transpose of weights + upsampling + extension (mw_upsample), then of the ring DFT
    const int mwss = P->sampling == SHT_MWSS, T2 = 4 * L;
    CK(st_adj_weight_pad(L, NBq, ldq, Fq, P->wq_quad, P->NB, T2, P->Z, st));
    CS(fft_exec(P, P->fft_th2, P->Z, P->Z, CUFFT_FORWARD, st));
    CK(st_adj_trunc_phase(L, mwss, P->NB, T2, P->Z, P->X, st));
    CS(fft_exec(P, P->fft_th1, P->X, P->X, CUFFT_INVERSE, st));
    CK(st_adj_fold(L, P->slab_n[0], mwss, P->NB, P->nrmap, P->F_ld, P->X, P->F, st));
    return fft_exec(P, P->fft_phi_inv, P->F, (double2*)f, CUFFT_INVERSE, st);
}

// ---- Wigner adjoints -------------------------------------------------------------------------------------------------
sht_status so3_forward_adjoint_plan(sht_plan* P, const void* flmn, void* f, sht_stream stream) {
    CS(check_ready(P));
    if (!flmn || !f || P->kind != 1) return SHT_EINVAL;
    if (P->sub.empty()) { g_err = "plan was not created with SHT_OPT_ADJOINT"; return SHT_EUNSUPPORTED; }
    cudaStream_t st = (cudaStream_t)stream;
    const size_t slab = (size_t)P->L * P->NB;
    for (int b = 0; b < P->nslab; ++b) {             // internal slabs are in gamma-FFT bin order, the coefficient array in n order
        const int n = P->slab_n[b];
        CK(st_scale_rows(P->L, P->M, (n & 1) ? -1.0 : 1.0, P->so3_dfwd, (const double2*)flmn + (size_t)(n + P->N - 1) * slab, P->adj_tmp, st));
        CS(s2_forward_adjoint_plan(P->sub[b], P->adj_tmp, (double2*)f + slab * b, stream));
    }
    return fft_exec(P, P->fft_gamma, (double2*)f, (double2*)f, CUFFT_INVERSE, st);      // transpose of f_n = sum_g f e^{-i n gamma_g}
}
sht_status so3_inverse_adjoint_plan(sht_plan* P, const void* f, void* flmn, sht_stream stream) {
    CS(check_ready(P));
    if (!flmn || !f || P->kind != 1) return SHT_EINVAL;
    if (P->sub.empty()) { g_err = "plan was not created with SHT_OPT_ADJOINT"; return SHT_EUNSUPPORTED; }
    cudaStream_t st = (cudaStream_t)stream;
    const size_t slab = (size_t)P->L * P->NB;
    CS(fft_exec(P, P->fft_gamma, (double2*)const_cast<void*>(f), P->fn, CUFFT_FORWARD, st));   // transpose of f = sum_n e^{+i n gamma_g} (...)
    for (int b = 0; b < P->nslab; ++b) {
        const int n = P->slab_n[b];
        CS(s2_inverse_adjoint_plan(P->sub[b], P->fn + slab * b, P->adj_tmp, stream));
        CK(st_scale_rows(P->L, P->M, (n & 1) ? -1.0 : 1.0, P->so3_dinv, P->adj_tmp, (double2*)flmn + (size_t)(n + P->N - 1) * slab, st));
    }
    return SHT_OK;
}

// ---- SO(3) (Eq. 15-18) ----------------------------------------------------------------------------
static sht_status so3_inverse_body(sht_plan* P, const void* flmn, void* f, sht_stream stream) {
    cudaStream_t st = (cudaStream_t)stream;
    const int L = P->L, NB = P->NB, N = P->N;
    const size_t slab = (size_t)L * NB;
    if (P->io_f32 && !P->f32_inner) {      // fp32 public arrays: fp64 copies around the core
        CK(st_f32_to_f64(2 * slab * P->nslab, (const float*)flmn, (double*)P->io_a, st));
        P->f32_inner = true;
        sht_status s = so3_inverse_body(P, P->io_a, P->io_b, stream);
        P->f32_inner = false;
        if (s != SHT_OK) return s;
        CK(st_f64_to_f32(2 * slab * P->nslab, (const double*)P->io_b, (float*)f, st));
        stage(P, CAT_STAGE, st);
        return SHT_OK;
    }
    begin_transform(P);
    stage(P, CAT_STAGE, st);
    // (coefficient slabs are read in place: the staging kernels map gamma-FFT bin order to n order through d_cslab)
    CS(run_theta_inverse(P, (const double2*)flmn, st));
    // F[n][bin][ring] -> f[n][ring][bin] (one transpose for all slabs), then the gamma transform (Eq. 17) and the ring synthesis of all
    // (gamma, beta) rows as ONE batched FFT each, in place in the output: 3 FFT launches instead of 2N per direction
    CK(st_transpose_slabs(P->nslab, NB, L, P->F_ld, NB, P->F, P->F_slab, (double2*)f, slab, st));
    stage(P, CAT_FFT, st);
    CS(fft_exec(P, P->fft_gamma, (double2*)f, (double2*)f, CUFFT_INVERSE, st));          // Eq. 17
    CS(fft_exec(P, P->fft_alpha, (double2*)f, (double2*)f, CUFFT_INVERSE, st));          // Eq. 32 on every row
    stage(P, CAT_STAGE, st);
    return SHT_OK;
}
static sht_status so3_forward_body(sht_plan* P, const void* f, void* flmn, sht_stream stream) {
    cudaStream_t st = (cudaStream_t)stream;
    const int L = P->L, NB = P->NB, N = P->N;
    const size_t slab = (size_t)L * NB;
    if (P->io_f32 && !P->f32_inner) {
        CK(st_f32_to_f64(2 * slab * P->nslab, (const float*)f, (double*)P->io_a, st));
        P->f32_inner = true;
        sht_status s = so3_forward_body(P, P->io_a, P->io_b, stream);
        P->f32_inner = false;
        if (s != SHT_OK) return s;
        CK(st_f64_to_f32(2 * slab * P->nslab, (const double*)P->io_b, (float*)flmn, st));
        stage(P, CAT_STAGE, st);
        return SHT_OK;
    }
    begin_transform(P);
    stage(P, CAT_FFT, st);
    CS(fft_exec(P, P->fft_gamma, (double2*)const_cast<void*>(f), P->fn, CUFFT_FORWARD, st));   // Eq. 16 (q_Gamma in scale_fwd)
    CS(fft_exec(P, P->fft_alpha, P->fn, P->fn, CUFFT_FORWARD, st));                            // ring DFTs of all (n, beta) rows, one batch
    stage(P, CAT_STAGE, st);
    CK(st_transpose_slabs(P->nslab, L, NB, NB, P->Ltp, P->fn, slab, P->Fa, P->Fa_slab, st));   // fn[n][ring][bin] -> Fa[n][bin][ring]
    CS(mw_upsample(P, st));
    CS(run_theta_forward(P, P->Z, (size_t)P->prow * P->fwd_ld, P->fwd_ld, st, P->pair));
    stage(P, CAT_STAGE, st);
    CK(st_finalize_forward(L, P->Lp, P->nslab, P->d_slab_n, P->d_cslab, 0, P->scale_fwd, P->H, P->H_slab, (double2*)flmn, slab, st));
    stage(P, CAT_STAGE, st);
    return SHT_OK;
}

}  // extern "C"

// ---- public transform calls: direct, or through a captured CUDA graph -----------------------------------------------------------
// At small band-limits a transform is a chain of 10-50 short launches (staging kernels, cuFFT passes, the fused kernels) and is bound
// by launch overhead, not by the GPU.  Plans with use_graph (default L <= 512; SHT_OPT_GRAPH / SHT_OPT_NO_GRAPH) capture the chain once
// per (direction, input pointer, output pointer) on an internal stream and replay it with ONE cudaGraphLaunch on the caller's stream.
// Stage timing, a caller that is itself capturing, and plans whose buffers change on every call (the cache misses) take the direct path.
namespace {
typedef sht_status (*transform_body)(sht_plan*, const void*, void*, sht_stream);
void drop_graphs(sht_plan* P) {
    for (auto& g : P->graphs) cudaGraphExecDestroy(g.exec);
    P->graphs.clear();
}
sht_status run_transform(sht_plan* P, int kind, const void* in, void* out, sht_stream stream, transform_body body) {
    cudaStream_t st = (cudaStream_t)stream;
    if (!P->use_graph || P->timing) return body(P, in, out, stream);
    cudaStreamCaptureStatus cst = cudaStreamCaptureStatusNone;
    if (cudaStreamIsCapturing(st, &cst) != cudaSuccess || cst != cudaStreamCaptureStatusNone) { (void)cudaGetLastError(); return body(P, in, out, stream); }
    for (auto& g : P->graphs)
        if (g.kind == kind && g.in == in && g.out == out) {
            CK(cudaGraphLaunch(g.exec, st));
            count_launch((int)g.launches);
            P->graph_hits++;
            return SHT_OK;
        }
    // buffers that change on every call would be re-captured every time: give up on graphs for this plan
    if (++P->graph_misses > 16 && P->graph_hits < P->graph_misses) { P->use_graph = false; drop_graphs(P); return body(P, in, out, stream); }
    if (!P->cap_stream) CK(cudaStreamCreateWithFlags(&P->cap_stream, cudaStreamNonBlocking));
    const long before = sht_launch_count(0);
    CK(cudaStreamBeginCapture(P->cap_stream, cudaStreamCaptureModeThreadLocal));
    sht_status s = body(P, in, out, (sht_stream)P->cap_stream);
    cudaGraph_t graph = nullptr;
    cudaError_t e = cudaStreamEndCapture(P->cap_stream, &graph);
    const long nl = sht_launch_count(0) - before;
    count_launch(-(int)nl);                                   // nothing ran yet
    if (s != SHT_OK || e != cudaSuccess || !graph) {
        if (graph) cudaGraphDestroy(graph);
        (void)cudaGetLastError();
        if (s != SHT_OK) return s;
        P->use_graph = false;                                 // capture not possible here: direct launches from now on
        return body(P, in, out, stream);
    }
    cudaGraphExec_t exec = nullptr;
    e = cudaGraphInstantiate(&exec, graph, 0);
    cudaGraphDestroy(graph);
    if (e != cudaSuccess) { (void)cudaGetLastError(); P->use_graph = false; return body(P, in, out, stream); }
    if (P->graphs.size() >= 8) { cudaGraphExecDestroy(P->graphs.front().exec); P->graphs.erase(P->graphs.begin()); }
    P->graphs.push_back({kind, in, out, exec, nl});
    CK(cudaGraphLaunch(exec, st));
    count_launch((int)nl);
    return SHT_OK;
}
}  // namespace

extern "C" {
// bytes of one map / one coefficient array of the public arrays (plans that run a batch map by map step through them)
static size_t map_bytes(const sht_plan* P) { return P->map_elems * (P->reality ? 1 : 2) * (P->io_f32 ? 4 : 8); }
static size_t coef_bytes(const sht_plan* P) { return (size_t)P->L * P->M * 2 * (P->io_f32 ? 4 : 8); }
sht_status s2_inverse_plan(sht_plan* P, const void* flm, void* f, sht_stream stream) {
    CS(check_ready(P));
    if (!flm || !f || P->kind != 0) return SHT_EINVAL;
    for (int b = 0; b < P->loop; ++b)
        CS(run_transform(P, 0, (const char*)flm + b * coef_bytes(P), (char*)f + b * map_bytes(P), stream, s2_inverse_body));
    return SHT_OK;
}
sht_status s2_forward_plan(sht_plan* P, const void* f, void* flm, sht_stream stream) {
    CS(check_ready(P));
    if (!flm || !f || P->kind != 0) return SHT_EINVAL;
    for (int b = 0; b < P->loop; ++b)
        CS(run_transform(P, 1, (const char*)f + b * map_bytes(P), (char*)flm + b * coef_bytes(P), stream, s2_forward_body));
    return SHT_OK;
}
sht_status so3_inverse_plan(sht_plan* P, const void* flmn, void* f, sht_stream stream) {
    CS(check_ready(P));
    if (!flmn || !f || P->kind != 1) return SHT_EINVAL;
    return run_transform(P, 0, flmn, f, stream, so3_inverse_body);
}
sht_status so3_forward_plan(sht_plan* P, const void* f, void* flmn, sht_stream stream) {
    CS(check_ready(P));
    if (!flmn || !f || P->kind != 1) return SHT_EINVAL;
    return run_transform(P, 1, f, flmn, stream, so3_forward_body);
}
}  // extern "C"

// ---- cached convenience calls ------------------------------------------------------------------------------------------

namespace {
// One entry per (device, problem).  The entry's mutex is held from lookup until the transform (and, for the *_host calls, the
// copies) have been enqueued, so two host threads never interleave on one plan's scratch; when consecutive calls use different
// streams, the new stream first waits for an event recorded after the previous call's work (one plan = one stream at a time).
struct CacheEntry {
    sht_plan* plan = nullptr; void* work = nullptr; void* d_in = nullptr; void* d_out = nullptr; size_t in_bytes = 0, out_bytes = 0;
    std::mutex mu; cudaEvent_t done = nullptr; cudaStream_t last = nullptr; bool used = false;
};
std::map<std::tuple<int, int, int, int, int, int, int>, CacheEntry*> g_cache;
std::mutex g_cache_mu;

struct CacheLease {
    CacheEntry* e = nullptr; cudaStream_t st = nullptr;
    std::unique_lock<std::mutex> lk;
    ~CacheLease() {
        if (!e) return;
        if (e->done) cudaEventRecord(e->done, st);
        e->last = st; e->used = true;
    }
};

sht_status cache_get(int kind, int L, int a, int sampling, int nside, int reality, cudaStream_t st, CacheLease* lease) {
    int dev = 0;
    CK(cudaGetDevice(&dev));
    CacheEntry* e = nullptr;
    {
        std::lock_guard<std::mutex> lk(g_cache_mu);
        auto key = std::make_tuple(dev, kind, L, a, sampling, nside, reality);
        auto it = g_cache.find(key);
        if (it == g_cache.end()) {
            sht_plan* plan = nullptr;
            sht_status s = kind == 0 ? sht_plan_s2(&plan, L, a, sampling, nside, reality, SHT_F64) : sht_plan_so3(&plan, L, a, SHT_F64);
            if (s != SHT_OK) return s;
            size_t nb = sht_plan_workspace_bytes(plan);
            void* work = nullptr;
            cudaError_t ce = cudaMalloc(&work, nb);
            if (ce != cudaSuccess) { g_err = std::string("cudaMalloc workspace: ") + cudaGetErrorString(ce); sht_plan_destroy(plan); return SHT_ECUDA; }
            s = sht_plan_set_workspace(plan, work, nb, st);
            if (s != SHT_OK) { cudaFree(work); sht_plan_destroy(plan); return s; }
            e = new CacheEntry();
            e->plan = plan; e->work = work;
            if (cudaEventCreateWithFlags(&e->done, cudaEventDisableTiming) != cudaSuccess) e->done = nullptr;
            it = g_cache.emplace(key, e).first;
        }
        e = it->second;
    }
    lease->lk = std::unique_lock<std::mutex>(e->mu);
    lease->e = e; lease->st = st;
    if (e->used && e->last != st && e->done) CK(cudaStreamWaitEvent(st, e->done, 0));
    return SHT_OK;
}
size_t s2_map_bytes(int L, int sampling, int nside, int reality) {
    size_t n;
    switch (sampling) {
        case SHT_HEALPIX: n = (size_t)12 * nside * nside; break;
        case SHT_MWSS: n = (size_t)(L + 1) * (2 * L); break;
        case SHT_DH: n = (size_t)(2 * L) * (2 * L - 1); break;
        default: n = (size_t)L * (2 * L - 1); break;
    }
    return n * (reality ? 8 : 16);
}
// copy stream and events of the chunked host-buffer calls (created on first use)
sht_status host_pipe_init(sht_plan* P) {
    if (P->copy_stream) return SHT_OK;
    CK(cudaStreamCreateWithFlags(&P->copy_stream, cudaStreamNonBlocking));
    for (auto& ev : P->ev_copy) CK(cudaEventCreateWithFlags(&ev, cudaEventDisableTiming));
    CK(cudaEventCreateWithFlags(&P->ev_begin, cudaEventDisableTiming));
    return SHT_OK;
}
sht_status host_io(CacheEntry* e, size_t in_bytes, size_t out_bytes) {
    if (e->in_bytes < in_bytes) { if (e->d_in) cudaFree(e->d_in); CK(cudaMalloc(&e->d_in, in_bytes)); e->in_bytes = in_bytes; }
    if (e->out_bytes < out_bytes) { if (e->d_out) cudaFree(e->d_out); CK(cudaMalloc(&e->d_out, out_bytes)); e->out_bytes = out_bytes; }
    return SHT_OK;
}
}  // namespace

extern "C" {

sht_status s2_forward(int L, int spin, int sampling, int reality, const void* f, void* flm, sht_stream stream) {
    CacheLease lease; CS(cache_get(0, L, spin, sampling, sampling == SHT_HEALPIX ? L / 2 : 0, reality, (cudaStream_t)stream, &lease));
    return s2_forward_plan(lease.e->plan, f, flm, stream);
}
sht_status s2_inverse(int L, int spin, int sampling, int reality, const void* flm, void* f, sht_stream stream) {
    CacheLease lease; CS(cache_get(0, L, spin, sampling, sampling == SHT_HEALPIX ? L / 2 : 0, reality, (cudaStream_t)stream, &lease));
    return s2_inverse_plan(lease.e->plan, flm, f, stream);
}
sht_status so3_forward(int L, int N, const void* f, void* flmn, sht_stream stream) {
    CacheLease lease; CS(cache_get(1, L, N, SHT_MW, 0, 0, (cudaStream_t)stream, &lease));
    return so3_forward_plan(lease.e->plan, f, flmn, stream);
}
sht_status so3_inverse(int L, int N, const void* flmn, void* f, sht_stream stream) {
    CacheLease lease; CS(cache_get(1, L, N, SHT_MW, 0, 0, (cudaStream_t)stream, &lease));
    return so3_inverse_plan(lease.e->plan, flmn, f, stream);
}
sht_status sht_cache_clear(void) {
    std::lock_guard<std::mutex> lk(g_cache_mu);
    for (auto& kv : g_cache) {
        CacheEntry* e = kv.second;
        { std::lock_guard<std::mutex> l2(e->mu); }
        sht_plan_destroy(e->plan);
        if (e->work) cudaFree(e->work);
        if (e->d_in) cudaFree(e->d_in);
        if (e->d_out) cudaFree(e->d_out);
        if (e->done) cudaEventDestroy(e->done);
        delete e;
    }
    g_cache.clear();
    return SHT_OK;
}

sht_status s2_forward_host(int L, int spin, int sampling, int reality, const void* f_host, void* flm_host, sht_stream stream) {
    cudaStream_t st = (cudaStream_t)stream;
    int nside = sampling == SHT_HEALPIX ? L / 2 : 0;
    CacheLease lease; CS(cache_get(0, L, spin, sampling, nside, reality, st, &lease));
    size_t mb = s2_map_bytes(L, sampling, nside, reality), cb = (size_t)L * (2 * L - 1) * 16;
    CacheEntry* e = lease.e; CS(host_io(e, mb > cb ? mb : cb, mb > cb ? mb : cb));
    sht_plan* P = e->plan;
    if (P->nchunk && !P->timing) {
        // ring chunks: the host -> device copy of chunk k+1 (copy stream) overlaps the ring FFT of chunk k (Eq. 31)
        CS(host_pipe_init(P));
        const size_t cbytes = mb / P->nchunk; const int crings = P->nrmap / P->nchunk;
        CK(cudaEventRecord(P->ev_begin, st)); CK(cudaStreamWaitEvent(P->copy_stream, P->ev_begin, 0));   // d_in is free once earlier work on st is done
        begin_transform(P);
        for (int k = 0; k < P->nchunk; ++k) {
            CK(cudaMemcpyAsync((char*)e->d_in + k * cbytes, (const char*)f_host + k * cbytes, cbytes, cudaMemcpyHostToDevice, P->copy_stream));
            CK(cudaEventRecord(P->ev_copy[k], P->copy_stream)); CK(cudaStreamWaitEvent(st, P->ev_copy[k], 0));
            CS(fft_exec(P, P->fft_phi_fwd_c, (double2*)((char*)e->d_in + k * cbytes), P->Fa + (size_t)k * crings, CUFFT_FORWARD, st));
        }
        P->skip_phi = true;
        sht_status s = s2_forward_plan(P, e->d_in, e->d_out, stream);
        P->skip_phi = false;
        CS(s);
    } else {
        CK(cudaMemcpyAsync(e->d_in, f_host, mb, cudaMemcpyHostToDevice, st));
        CS(s2_forward_plan(P, e->d_in, e->d_out, stream));
    }
    CK(cudaMemcpyAsync(flm_host, e->d_out, cb, cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    return SHT_OK;
}
sht_status s2_inverse_host(int L, int spin, int sampling, int reality, const void* flm_host, void* f_host, sht_stream stream) {
    cudaStream_t st = (cudaStream_t)stream;
    int nside = sampling == SHT_HEALPIX ? L / 2 : 0;
    CacheLease lease; CS(cache_get(0, L, spin, sampling, nside, reality, st, &lease));
    size_t mb = s2_map_bytes(L, sampling, nside, reality), cb = (size_t)L * (2 * L - 1) * 16;
    CacheEntry* e = lease.e; CS(host_io(e, mb > cb ? mb : cb, mb > cb ? mb : cb));
    CK(cudaMemcpyAsync(e->d_in, flm_host, cb, cudaMemcpyHostToDevice, st));
    sht_plan* P = e->plan;
    if (P->nchunk && !P->timing) {
        // ring chunks: the device -> host copy of chunk k (copy stream) overlaps the ring synthesis of chunk k+1 (Eq. 32)
        CS(host_pipe_init(P));
        const size_t cbytes = mb / P->nchunk; const int crings = P->nrmap / P->nchunk;
        P->skip_phi = true;
        sht_status s = s2_inverse_plan(P, e->d_in, e->d_out, stream);
        P->skip_phi = false;
        CS(s);
        for (int k = 0; k < P->nchunk; ++k) {
            CS(fft_exec(P, P->fft_phi_inv_c, P->F + (size_t)k * crings, (double2*)((char*)e->d_out + k * cbytes), CUFFT_INVERSE, st));
            CK(cudaEventRecord(P->ev_copy[k], st)); CK(cudaStreamWaitEvent(P->copy_stream, P->ev_copy[k], 0));
            CK(cudaMemcpyAsync((char*)f_host + k * cbytes, (char*)e->d_out + k * cbytes, cbytes, cudaMemcpyDeviceToHost, P->copy_stream));
        }
        CK(cudaStreamSynchronize(P->copy_stream));
    } else {
        CS(s2_inverse_plan(P, e->d_in, e->d_out, stream));
        CK(cudaMemcpyAsync(f_host, e->d_out, mb, cudaMemcpyDeviceToHost, st));
    }
    CK(cudaStreamSynchronize(st));
    return SHT_OK;
}
sht_status so3_forward_host(int L, int N, const void* f_host, void* flmn_host, sht_stream stream) {
    cudaStream_t st = (cudaStream_t)stream;
    CacheLease lease; CS(cache_get(1, L, N, SHT_MW, 0, 0, st, &lease));
    size_t b = (size_t)(2 * N - 1) * L * (2 * L - 1) * 16;
    CacheEntry* e = lease.e; CS(host_io(e, b, b));
    CK(cudaMemcpyAsync(e->d_in, f_host, b, cudaMemcpyHostToDevice, st));
    CS(so3_forward_plan(e->plan, e->d_in, e->d_out, stream));
    CK(cudaMemcpyAsync(flmn_host, e->d_out, b, cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    return SHT_OK;
}
sht_status so3_inverse_host(int L, int N, const void* flmn_host, void* f_host, sht_stream stream) {
    cudaStream_t st = (cudaStream_t)stream;
    CacheLease lease; CS(cache_get(1, L, N, SHT_MW, 0, 0, st, &lease));
    size_t b = (size_t)(2 * N - 1) * L * (2 * L - 1) * 16;
    CacheEntry* e = lease.e; CS(host_io(e, b, b));
    CK(cudaMemcpyAsync(e->d_in, flmn_host, b, cudaMemcpyHostToDevice, st));
    CS(so3_inverse_plan(e->plan, e->d_in, e->d_out, stream));
    CK(cudaMemcpyAsync(f_host, e->d_out, b, cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    return SHT_OK;
}

sht_status sht_peak(int kind, int iters, double* tflops, float* ms, sht_stream stream) {
    if (!tflops || !ms || iters < 1 || kind < 0 || kind > 3) return SHT_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    int dev = 0, nsm = 0;
    CK(cudaGetDevice(&dev));
    CK(cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev));
    double* sink = nullptr;
    CK(cudaMalloc(&sink, 8));
    cudaEvent_t a, b;
    CK(cudaEventCreate(&a)); CK(cudaEventCreate(&b));
    double flop = 0;
    CK(launch_peak(kind, iters / 8 + 1, nsm, sink, st, &flop));       // warm-up
    CK(cudaEventRecord(a, st));
    CK(launch_peak(kind, iters, nsm, sink, st, &flop));
    CK(cudaEventRecord(b, st));
    CK(cudaEventSynchronize(b));
    CK(cudaEventElapsedTime(ms, a, b));
    *tflops = flop / (*ms * 1e-3) / 1e12;
    cudaEventDestroy(a); cudaEventDestroy(b); cudaFree(sink);
    return SHT_OK;
}
sht_status sht_fp64_peak(int iters, double* tflops, float* ms, sht_stream stream) { return sht_peak(SHT_PEAK_DFMA, iters, tflops, ms, stream); }

}  // extern "C"
