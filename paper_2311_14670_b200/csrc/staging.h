// staging.h -- launchers of the table-setup and staging kernels (staging.cu).  Internal.
#pragma once
#include "internal.h"

cudaError_t st_start_values(int L, int n, int nth, int ntp, const double* c2hi, const double* c2lo, const double* s2hi,
                            const double* s2lo, const double* rhi, const double* rlo, double* st_val, uint8_t* st_k, int* range_flag,
                            cudaStream_t st);
cudaError_t st_kexp(int nrows, int kstride, int kmin, int8_t* kexp, cudaStream_t st);
cudaError_t st_rsq(int n, double* rsq, cudaStream_t st);
cudaError_t st_mw_weights(int Lq, double qphi, double* w, cudaStream_t st);
cudaError_t st_mid_weights(int L, int count, double qphi, double* w, cudaStream_t st);
cudaError_t st_prep_inverse(int L, int Lp, int NC, int mmin, int npass, const double2* coef, size_t coef_slab, const int* cslab,
                            const double* scale, const double* C, const double2* SG, int sgstride, const ThetaPass* passes, cudaStream_t st);
cudaError_t st_ctab(int L, int Lp, int mmin, int kstride, int kmin, const int8_t* kexp, const double* rsq, double* C, cudaStream_t st);
cudaError_t st_sgtab(int nrows, int ncol, int mmin, int kstride, int kmin, const int8_t* kexp, double2* SG, cudaStream_t st);
cudaError_t st_lamtab(int n, int nth, int ntp, int m_end, int nrows, const double* csc, const double* tau, const double* sig, double* lam,
                      cudaStream_t st);
cudaError_t st_pole_inverse(int L, int north, int NBf, int nslab, const int* slab_n, const int* cslab, const double2* coef, size_t coef_slab,
                            const double* scale, double2* F, size_t F_slab, int ldf, int col, cudaStream_t st);
cudaError_t st_hermitian_rows(int L, int NB, int ntp, int nth, double2* F, cudaStream_t st);
cudaError_t st_real_to_complex(size_t n, const double* in, double2* out, cudaStream_t st);
cudaError_t st_complex_to_real(size_t n, const double2* in, double* out, cudaStream_t st);
cudaError_t st_mw_extend(int L, int nslab, const int* slab_n, int mwss, int pair, int ldin, int ldout, const double2* Fa, size_t Fa_slab, double2* X,
                         size_t X_slab, cudaStream_t st);
cudaError_t st_mw_pad_phase(int L, int nslab, int mwss, int rows, int ldin, int ldout, const double2* Y, size_t Y_slab, double2* Z, size_t Z_slab,
                            cudaStream_t st);
cudaError_t st_weight_split(int L, int NBin, int ldin, int pair, int nth, int ntp, int NC, int mmin, int npass, const double* wq, const double2* U,
                            size_t U_slab, const ThetaPass* passes, int th_lo, int th_hi, cudaStream_t st);
cudaError_t st_weight_split_fold0(int L, int NBin, int ldin, int pair, int nth, int ntp, int nfull, int NC, int m_end, const double* wq,
                                  const double2* U, double2* W, int th_lo, int th_hi, cudaStream_t st);
cudaError_t st_pole_forward(int L, int Lp, int n, int north, int NBin, int ldin, int col, double w, const double2* U, double2* H,
                            cudaStream_t st);
cudaError_t st_finalize_forward(int L, int Lp, int nslab, const int* slab_n, const int* cslab, int real, const double* scale, const double2* H,
                                size_t H_slab, double2* coef, size_t coef_slab, cudaStream_t st);
cudaError_t st_rows_reorder(int L, int NB, int ncol, int ldsrc, int lddst, int to_mi, const double2* src, double2* dst, cudaStream_t st);
cudaError_t st_scale_copy(size_t n, double s, const double2* in, double2* out, cudaStream_t st);

// adjoint transforms: conjugate transposes of the staging steps (Sec. 5.3)
cudaError_t st_scale_cols(int nrows, int ncol, int ld, const double* w, double2* F, cudaStream_t st);
cudaError_t st_adj_weight_pad(int L, int NBq, int ldq, const double2* Fq, const double* wq, int NB, int T2, double2* Z, cudaStream_t st);
cudaError_t st_adj_trunc_phase(int L, int mwss, int NB, int T2, const double2* Zf, double2* X, cudaStream_t st);
cudaError_t st_adj_fold(int L, int n, int mwss, int NB, int nrmap, int ldf, const double2* X, double2* F, cudaStream_t st);

// HEALPix iterative refinement: out = a - b; y += x (arrays of doubles)
cudaError_t st_vec_sub(size_t n, const double* a, const double* b, double* out, cudaStream_t st);
cudaError_t st_vec_add(size_t n, const double* x, double* y, cudaStream_t st);

// MW inverse through the symmetric midpoint rings: resampling of F_m to the MW rings
cudaError_t st_sym_extend(int L, int n, int pair, int ldin, const double2* F, double2* X, cudaStream_t st);
cudaError_t st_sym_rebin(int L, int rows, const double2* Y, double2* Z, cudaStream_t st);
cudaError_t st_sym_unpair(int L, int n, int ldout, const double2* X, double2* F, cudaStream_t st);
cudaError_t st_scale_rows(int nrow, int ncol, double sgn, const double* d, const double2* in, double2* out, cudaStream_t st);
cudaError_t st_transpose_slabs(int nslab, int nrow, int ncol, int ldin, int ldout, const double2* in, size_t in_slab, double2* out,
                               size_t out_slab, cudaStream_t st);
cudaError_t st_rows_head(int nrows, int ncol, int ldin, int ldout, const double2* in, double2* out, cudaStream_t st);

// batched path (operand / result layouts of theta_mma.cu, internal.h)
cudaError_t st_prep_inverse_batch(int L, int Lp, int NC, int B, int ncg, int n, int sgn_out, int m_end, int mmin, const double2* coef,
                                  const double* scale, const double* C, const double2* SG, int sgstride, double* Gb, size_t cg_stride,
                                  cudaStream_t st);
cudaError_t st_weight_split_batch(int L, int NBin, int ldin, int pair, size_t U_slab, int nth, int ntp, int NC, int B, int ncg, int n, int sgn_out,
                                  int m_end, int fold, const int* m_lo, const double* wq, const double* lam, const double2* U, double* Wb,
                                  size_t cg_stride, cudaStream_t st);
cudaError_t st_weight_split_batch_fold0(int L, int NBin, int ldin, int pair, size_t U_slab, int nth, int ntp, int nfull, int NC, int B, int ncg,
                                        int m_end, const double* wq, const double* lam, const double2* U, double* Wb, size_t cg_stride,
                                        cudaStream_t st);
cudaError_t st_unpack_batch(int L, int Lp, int Mp, int mlim, int NC, int B, int ncg, int n, int sgn_out, int m_end, int mmin, int fwd, int fold,
                            const double* C, const double* Ob, size_t cg_stride, double2* out, size_t out_slab, int ld, cudaStream_t st);

// fp32 variant (theta_f32.cu): tables, operand preparation, precision conversion of the public arrays
cudaError_t st_ab32(int L, int Lp, float4* AB, cudaStream_t st);
cudaError_t st_start32(size_t n, const double* v64, const uint8_t* k64, float* v32, uint16_t* k16, cudaStream_t st);
cudaError_t st_prep_inverse_f32(int L, int Lp, int NC, const double2* coef, const double* scale, float2* G, cudaStream_t st);
cudaError_t st_weight_split_f32(int L, int NBin, int ldin, int pair, int nth, int ntp, int NC, const double* wq, const double2* U, float2* W,
                                cudaStream_t st);
cudaError_t st_weight_split_f32_fold0(int L, int NBin, int ldin, int pair, int nth, int ntp, int nfull, int NC, const double* wq, const double2* U,
                                      float2* W, cudaStream_t st);
cudaError_t st_f32_to_f64(size_t n, const float* in, double* out, cudaStream_t st);
cudaError_t st_f64_to_f32(size_t n, const double* in, float* out, cudaStream_t st);

// HEALPix ring Fourier staging (healpix.cu)
void hp_ring_host(int nside, int i, int* nphi, int* shifted, long long* off);
cudaError_t st_hp_chirp(int nside, int M, double2* BF, cudaStream_t st);
cudaError_t st_hp_pack_fwd(int nside, int M, int real_in, const void* map, double2* C, cudaStream_t st);
cudaError_t st_hp_mul(int nside, int M, const double2* BF, double2* C, cudaStream_t st);
cudaError_t st_hp_unpack_fwd(int nside, int L, int NB, int mlo, int ldu, int M, const double2* C, const double2* E, double2* U,
                             cudaStream_t st);
cudaError_t st_hp_fold_inv(int nside, int L, int NB, int ldf, int M, const double2* F, double2* C, double2* E, cudaStream_t st);
cudaError_t st_hp_unpack_inv(int nside, int M, int real_out, const double2* C, void* map, cudaStream_t st);
cudaError_t st_hp_belt_real(size_t n, const double2* E, double* out, cudaStream_t st);
