/*
 * holo_oracle.h -- CPU oracle for the hot path of arXiv 2004.00923
 * ("Real-time digital holography of the retina by principal component analysis").
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may load it.  It shares no code,
 * header, table or helper with the CUDA path under paper_2004_00923_b200/csrc/.
 *
 * Everything is the plain definition, in double precision, in the paper's order:
 *   d_t   = I_t - mean_t I                                  (BASELINE.json north_star)
 *   g_t   = d_t * exp(+i*pi*(x^2+y^2)/(lambda z))           (Eq. 1 expanded;
 *                                                            sign/centre: DESIGN.md readings R3,R6)
 *   H_t   = unnormalised forward 2-D DFT of g_t             ("one spatial Fourier transform")
 *   C     = H^{t*} H   (T x T, sum over all pixels)         (Eq. 4)
 *   C     = V Lambda V^{t*}                                 (Eq. 5)
 *   Hc    = H V I_f                                         (Eq. 6)
 *   M     = sum_{k in [k_lo,k_hi]} |Hc_k|^2                 (Eq. 7)
 *   Ht    = H W I_f,  M0 = sum |Ht|^2                       (Eq. 8-9)
 *   Hf    = U Delta I_f V^{t*} = H V I_f V^{t*}             (Eq. 3: SVD filter)
 *   Mn    = M / <M>   (division by the spatial average)
 *   shift = quadrant swap of an image in FFT-bin order      (display convention, R6)
 *
 * Pins (tests/test_oracle_*.py, all "-m not gpu"): brute-force DFT, Parseval, point-source
 * closed forms, exact integer Gram, 2x2 closed form, T=2 closed form, LAPACK eigh/svd on tiny
 * inputs, energy conservation, pure-tone <-> DFT-basis equivalence.  No function here is
 * "parity unpinned".
 *
 * Layouts: complex arrays are interleaved (re,im) doubles.
 *   frames  uint16 [T][ny][nx]        H  complex [T][ny*nx]
 *   C       complex [T][T] row-major  V  complex [T][T] row-major, column k-1 = eigenvector k
 *   evals   double [T] DESCENDING (k = 1 is the largest; reading R1)
 *   P       complex [T][ny*nx] (component-planar), M double [ny*nx]
 */
#ifndef HOLO_ORACLE_H
#define HOLO_ORACLE_H
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

/* In-place unnormalised forward 2-D DFT (e^{-2 pi i ...}) of one ny x nx complex image,
 * own iterative radix-2 Cooley-Tukey, rows then columns.  nx, ny powers of two. Returns 0 / -1. */
int oracle_fft2(double* data, int ny, int nx);

/* chirp q(i,j) = exp(+i pi (x_i^2 + y_j^2)/(lambda z)), x_i = (i-nx/2) pitch, y_j = (j-ny/2) pitch */
int oracle_chirp(int nx, int ny, double lambda_m, double pitch_m, double z_m, double* q);

/* d_t = I_t - mean_t I  (double [T][ny*nx]) */
int oracle_mean_subtract(const uint16_t* frames, int nx, int ny, int T, double* d);

/* frames -> H (steps 1-3) */
int oracle_fresnel(const uint16_t* frames, int nx, int ny, int T,
                   double lambda_m, double pitch_m, double z_m, double* H);

/* Fresnel hologram of an arbitrary complex field g (no mean subtraction): H = FFT2[g*q]; pin helper */
int oracle_fresnel_field(const double* g, int nx, int ny,
                         double lambda_m, double pitch_m, double z_m, double* H);

/* C_ts = sum_p conj(H_t(p)) H_s(p), direct sums */
int oracle_covariance(const double* H, long long n_pix, int T, double* C);

/* cyclic-by-row complex Hermitian Jacobi; descending order; returns sweeps used (>=0) or -1 */
int oracle_eig(const double* C, int T, double* evals, double* V);

/* P_k(p) = sum_t H_t(p) V_{t,k}, all k = 1..T */
int oracle_project(const double* H, long long n_pix, int T, const double* V, double* P);

/* M(p) = sum_{k=k_lo}^{k_hi} |P_k(p)|^2  (1-based inclusive) */
int oracle_envelope(const double* P, long long n_pix, int T, int k_lo, int k_hi, double* M);

/* Eq. 8: W_{mn} = exp(-2 i pi (m-1)(n-1)/T)/sqrt(T), row-major [T][T] */
int oracle_dft_basis(int T, double* W);

/* whole path; any of H_out, C_out, evals_out, V_out may be NULL */
int oracle_process(const uint16_t* frames, int nx, int ny, int T,
                   double lambda_m, double pitch_m, double z_m, int k_lo, int k_hi,
                   double* M, double* H_out, double* C_out, double* evals_out, double* V_out);

/* Eq. 3: Hf = H V I_f V^{t*}: project on all components, keep k_lo..k_hi (1-based inclusive,
 * descending order), come back to the frame basis.  Hf complex [T][n_pix]. */
int oracle_svd_filter(const double* H, long long n_pix, int T, const double* V, int k_lo, int k_hi, double* Hf);

/* PAPER.md:86 ("image normalization by their respective average value"): out(p) = M(p) / ((1/n_pix) sum_p M(p)).
 * A zero image is returned unchanged. */
int oracle_normalize(const double* M, long long n_pix, double* out);

/* Quadrant swap: out[(j + ny/2) mod ny][(i + nx/2) mod nx] = in[j][i]  (zero frequency to the centre). */
int oracle_fftshift(const double* in, int ny, int nx, double* out);

int oracle_num_threads(void);

#ifdef __cplusplus
}
#endif
#endif
