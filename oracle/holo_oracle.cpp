// holo_oracle.cpp -- CPU oracle (double precision) for arXiv 2004.00923's hot path.
// TEST INFRASTRUCTURE ONLY; see holo_oracle.h for scope, citations and pins.
// Shares nothing with the CUDA path.  OpenMP is used only over independent outer loops.
#include "holo_oracle.h"
#include <cmath>
#include <complex>
#include <vector>
#include <algorithm>
#include <numeric>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef std::complex<double> cd;
static const double PI = 3.14159265358979323846264338327950288;

static bool is_pow2(int n) { return n >= 1 && (n & (n - 1)) == 0; }

// ---------------------------------------------------------------------------------------------
// 1-D FFT: iterative radix-2 Cooley-Tukey, decimation in time, forward sign e^{-2 pi i nk/N},
// unnormalised (reading R5; "one spatial Fourier transform", cuFFT).
// x has `n` elements at stride `stride`.
// ---------------------------------------------------------------------------------------------
static void fft1d(cd* x, int n, long long stride, const std::vector<cd>& w /* w[k]=e^{-2 pi i k/n}, k<n/2 */) {
    // bit reversal permutation
    for (int i = 1, j = 0; i < n; ++i) {
        int bit = n >> 1;
        for (; j & bit; bit >>= 1) j ^= bit;
        j ^= bit;
        if (i < j) std::swap(x[i * stride], x[j * stride]);
    }
    for (int len = 2; len <= n; len <<= 1) {
        int half = len >> 1, step = n / len;
        for (int base = 0; base < n; base += len) {
            for (int k = 0; k < half; ++k) {
                cd u = x[(base + k) * stride];
                cd v = x[(base + k + half) * stride] * w[k * step];
                x[(base + k) * stride] = u + v;
                x[(base + k + half) * stride] = u - v;
            }
        }
    }
}

static std::vector<cd> twiddles(int n) {
    std::vector<cd> w(std::max(1, n / 2));
    for (int k = 0; k < n / 2; ++k) {
        double a = -2.0 * PI * (double)k / (double)n;
        w[k] = cd(std::cos(a), std::sin(a));
    }
    return w;
}

static void fft2_inplace(cd* a, int ny, int nx) {
    std::vector<cd> wx = twiddles(nx), wy = twiddles(ny);
    for (int j = 0; j < ny; ++j) fft1d(a + (long long)j * nx, nx, 1, wx);   // rows (over x)
    for (int i = 0; i < nx; ++i) fft1d(a + i, ny, nx, wy);                  // columns (over y)
}

extern "C" int oracle_fft2(double* data, int ny, int nx) {
    if (!data || !is_pow2(nx) || !is_pow2(ny)) return -1;
    fft2_inplace(reinterpret_cast<cd*>(data), ny, nx);
    return 0;
}

// ---------------------------------------------------------------------------------------------
// chirp: q(i,j) = exp(+i pi (x_i^2 + y_j^2)/(lambda z)), centred integer offsets (R3, R6).
// Evaluated directly from the formula at every pixel (no separable table: that is the GPU's trick).
// ---------------------------------------------------------------------------------------------
extern "C" int oracle_chirp(int nx, int ny, double lambda_m, double pitch_m, double z_m, double* q_) {
    if (!q_ || nx < 1 || ny < 1 || !(lambda_m > 0) || !(pitch_m > 0) || !(z_m > 0)) return -1;
    cd* q = reinterpret_cast<cd*>(q_);
    for (int j = 0; j < ny; ++j) {
        double y = (double)(j - ny / 2) * pitch_m;
        for (int i = 0; i < nx; ++i) {
            double x = (double)(i - nx / 2) * pitch_m;
            double ph = PI * (x * x + y * y) / (lambda_m * z_m);
            q[(long long)j * nx + i] = cd(std::cos(ph), std::sin(ph));
        }
    }
    return 0;
}

// d_t = I_t - (1/T) sum_s I_s, per pixel, over the T frames of this stack (reading R2).
extern "C" int oracle_mean_subtract(const uint16_t* frames, int nx, int ny, int T, double* d) {
    if (!frames || !d || nx < 1 || ny < 1 || T < 1) return -1;
    long long np = (long long)nx * ny;
    for (long long p = 0; p < np; ++p) {
        double s = 0.0;
        for (int t = 0; t < T; ++t) s += (double)frames[(long long)t * np + p];
        double mean = s / (double)T;
        for (int t = 0; t < T; ++t) d[(long long)t * np + p] = (double)frames[(long long)t * np + p] - mean;
    }
    return 0;
}

extern "C" int oracle_fresnel_field(const double* g_, int nx, int ny,
                                    double lambda_m, double pitch_m, double z_m, double* H_) {
    if (!g_ || !H_ || !is_pow2(nx) || !is_pow2(ny)) return -1;
    long long np = (long long)nx * ny;
    std::vector<cd> q(np);
    if (oracle_chirp(nx, ny, lambda_m, pitch_m, z_m, reinterpret_cast<double*>(q.data()))) return -1;
    const cd* g = reinterpret_cast<const cd*>(g_);
    cd* H = reinterpret_cast<cd*>(H_);
    for (long long p = 0; p < np; ++p) H[p] = g[p] * q[p];
    fft2_inplace(H, ny, nx);
    return 0;
}

extern "C" int oracle_fresnel(const uint16_t* frames, int nx, int ny, int T,
                              double lambda_m, double pitch_m, double z_m, double* H_) {
    if (!frames || !H_ || !is_pow2(nx) || !is_pow2(ny) || T < 1) return -1;
    long long np = (long long)nx * ny;
    std::vector<double> d((size_t)T * np);
    if (oracle_mean_subtract(frames, nx, ny, T, d.data())) return -1;
    std::vector<cd> q(np);
    if (oracle_chirp(nx, ny, lambda_m, pitch_m, z_m, reinterpret_cast<double*>(q.data()))) return -1;
    cd* H = reinterpret_cast<cd*>(H_);
#pragma omp parallel for schedule(static)
    for (int t = 0; t < T; ++t) {
        cd* Ht = H + (long long)t * np;
        for (long long p = 0; p < np; ++p) Ht[p] = d[(long long)t * np + p] * q[p];
        fft2_inplace(Ht, ny, nx);
    }
    return 0;
}

// ---------------------------------------------------------------------------------------------
// Eq. 4: C = H^{t*} H, C_ts = sum_p conj(H_t(p)) H_s(p); no normalisation (R9).
// Every (t,s) entry is its own direct sum (no Hermitian shortcut: the definition, written out).
// ---------------------------------------------------------------------------------------------
extern "C" int oracle_covariance(const double* H_, long long n_pix, int T, double* C_) {
    if (!H_ || !C_ || n_pix < 0 || T < 1) return -1;
    const cd* H = reinterpret_cast<const cd*>(H_);
    cd* C = reinterpret_cast<cd*>(C_);
#pragma omp parallel for schedule(dynamic)
    for (int ts = 0; ts < T * T; ++ts) {
        int t = ts / T, s = ts % T;
        const cd* Ht = H + (long long)t * n_pix;
        const cd* Hs = H + (long long)s * n_pix;
        cd acc(0.0, 0.0);
        for (long long p = 0; p < n_pix; ++p) acc += std::conj(Ht[p]) * Hs[p];
        C[ts] = acc;
    }
    return 0;
}

// ---------------------------------------------------------------------------------------------
// Eq. 5: C = V Lambda V^{t*}.  Cyclic-by-row complex Hermitian Jacobi.
// Pivot (p,q), a_pq = |a_pq| e^{i phi}:  tau = (a_qq - a_pp)/(2|a_pq|),
//   t = sgn(tau)/(|tau| + sqrt(1+tau^2)),  c = 1/sqrt(1+t^2),  s = t c,
//   J = [[c, s e^{i phi}], [-s e^{-i phi}, c]] on rows/cols (p,q);  A <- J^H A J,  V <- V J.
// Stops when sqrt(sum_{p!=q}|a_pq|^2) <= 1e-14 ||C||_F.  Output sorted DESCENDING (R1).
// ---------------------------------------------------------------------------------------------
extern "C" int oracle_eig(const double* C_, int T, double* evals, double* V_) {
    if (!C_ || !evals || !V_ || T < 1) return -1;
    const cd* C = reinterpret_cast<const cd*>(C_);
    std::vector<cd> A(C, C + (size_t)T * T), V((size_t)T * T, cd(0, 0));
    for (int i = 0; i < T; ++i) V[i * T + i] = 1.0;
    // symmetrise the input to exactly Hermitian (the input is Hermitian up to rounding)
    for (int i = 0; i < T; ++i) {
        A[i * T + i] = cd(A[i * T + i].real(), 0.0);
        for (int j = i + 1; j < T; ++j) {
            cd m = 0.5 * (A[i * T + j] + std::conj(A[j * T + i]));
            A[i * T + j] = m; A[j * T + i] = std::conj(m);
        }
    }
    double normF = 0.0;
    for (size_t i = 0; i < A.size(); ++i) normF += std::norm(A[i]);
    normF = std::sqrt(normF);
    int sweeps = 0;
    const int max_sweeps = 60;
    for (; sweeps < max_sweeps; ++sweeps) {
        double off = 0.0;
        for (int p = 0; p < T; ++p) for (int q = 0; q < T; ++q) if (p != q) off += std::norm(A[p * T + q]);
        if (std::sqrt(off) <= 1e-14 * normF) break;
        for (int p = 0; p < T - 1; ++p) {
            for (int q = p + 1; q < T; ++q) {
                cd apq = A[p * T + q];
                double mag = std::abs(apq);
                double app = A[p * T + p].real(), aqq = A[q * T + q].real();
                if (mag <= 1e-300 || mag <= 1e-17 * std::sqrt(std::fabs(app * aqq))) continue;
                cd eiphi = apq / mag;                       // e^{i phi}
                double tau = (aqq - app) / (2.0 * mag), t;
                if (std::fabs(tau) > 1e8) t = 1.0 / (2.0 * tau);
                else t = (tau >= 0 ? 1.0 : -1.0) / (std::fabs(tau) + std::sqrt(1.0 + tau * tau));
                double c = 1.0 / std::sqrt(1.0 + t * t), s = t * c;
                cd se = s * eiphi, sec = s * std::conj(eiphi);  // s e^{i phi}, s e^{-i phi}
                for (int i = 0; i < T; ++i) {                // A <- A J  (columns p,q)
                    cd ap = A[i * T + p], aq = A[i * T + q];
                    A[i * T + p] = c * ap - sec * aq;
                    A[i * T + q] = se * ap + c * aq;
                }
                for (int j = 0; j < T; ++j) {                // A <- J^H A  (rows p,q)
                    cd ap = A[p * T + j], aq = A[q * T + j];
                    A[p * T + j] = c * ap - se * aq;
                    A[q * T + j] = sec * ap + c * aq;
                }
                for (int i = 0; i < T; ++i) {                // V <- V J
                    cd vp = V[i * T + p], vq = V[i * T + q];
                    V[i * T + p] = c * vp - sec * vq;
                    V[i * T + q] = se * vp + c * vq;
                }
                A[p * T + q] = 0.0; A[q * T + p] = 0.0;
                A[p * T + p] = cd(A[p * T + p].real(), 0.0);
                A[q * T + q] = cd(A[q * T + q].real(), 0.0);
            }
        }
    }
    std::vector<int> order(T);
    std::iota(order.begin(), order.end(), 0);
    std::stable_sort(order.begin(), order.end(),
                     [&](int a, int b) { return A[a * T + a].real() > A[b * T + b].real(); });
    cd* Vout = reinterpret_cast<cd*>(V_);
    for (int k = 0; k < T; ++k) {
        evals[k] = A[order[k] * T + order[k]].real();
        for (int i = 0; i < T; ++i) Vout[i * T + k] = V[i * T + order[k]];
    }
    return sweeps;
}

// Eq. 6: Hc = H V, P_k(p) = sum_t H_t(p) V_{t,k}; all k so invariants can be checked.
extern "C" int oracle_project(const double* H_, long long n_pix, int T, const double* V_, double* P_) {
    if (!H_ || !V_ || !P_ || T < 1 || n_pix < 0) return -1;
    const cd* H = reinterpret_cast<const cd*>(H_);
    const cd* V = reinterpret_cast<const cd*>(V_);
    cd* P = reinterpret_cast<cd*>(P_);
#pragma omp parallel for schedule(static)
    for (int k = 0; k < T; ++k) {
        cd* Pk = P + (long long)k * n_pix;
        for (long long p = 0; p < n_pix; ++p) {
            cd acc(0, 0);
            for (int t = 0; t < T; ++t) acc += H[(long long)t * n_pix + p] * V[t * T + k];
            Pk[p] = acc;
        }
    }
    return 0;
}

// Eq. 7: M(p) = sum_{k=k_lo}^{k_hi} |P_k(p)|^2, 1-based inclusive (R13).
extern "C" int oracle_envelope(const double* P_, long long n_pix, int T, int k_lo, int k_hi, double* M) {
    if (!P_ || !M || k_lo < 1 || k_hi > T || k_lo > k_hi) return -1;
    const cd* P = reinterpret_cast<const cd*>(P_);
    for (long long p = 0; p < n_pix; ++p) {
        double acc = 0.0;
        for (int k = k_lo; k <= k_hi; ++k) acc += std::norm(P[(long long)(k - 1) * n_pix + p]);
        M[p] = acc;
    }
    return 0;
}

// Eq. 8: w_mn = exp(-2 i (m-1)(n-1) pi / n_t)/sqrt(n_t), m,n = 1..n_t
extern "C" int oracle_dft_basis(int T, double* W_) {
    if (!W_ || T < 1) return -1;
    cd* W = reinterpret_cast<cd*>(W_);
    for (int m = 1; m <= T; ++m)
        for (int n = 1; n <= T; ++n) {
            double a = -2.0 * (double)(m - 1) * (double)(n - 1) * PI / (double)T;
            W[(m - 1) * T + (n - 1)] = cd(std::cos(a), std::sin(a)) / std::sqrt((double)T);
        }
    return 0;
}

extern "C" int oracle_process(const uint16_t* frames, int nx, int ny, int T,
                              double lambda_m, double pitch_m, double z_m, int k_lo, int k_hi,
                              double* M, double* H_out, double* C_out, double* evals_out, double* V_out) {
    if (!frames || !M || k_lo < 1 || k_hi > T || k_lo > k_hi) return -1;
    long long np = (long long)nx * ny;
    std::vector<double> Hbuf, P((size_t)2 * T * np), C((size_t)2 * T * T), V((size_t)2 * T * T), ev(T);
    double* H = H_out;
    if (!H) { Hbuf.resize((size_t)2 * T * np); H = Hbuf.data(); }
    if (oracle_fresnel(frames, nx, ny, T, lambda_m, pitch_m, z_m, H)) return -1;
    if (oracle_covariance(H, np, T, C.data())) return -1;
    int sw = oracle_eig(C.data(), T, ev.data(), V.data());
    if (sw < 0) return -1;
    if (oracle_project(H, np, T, V.data(), P.data())) return -1;
    if (oracle_envelope(P.data(), np, T, k_lo, k_hi, M)) return -1;
    if (C_out) std::copy(C.begin(), C.end(), C_out);
    if (V_out) std::copy(V.begin(), V.end(), V_out);
    if (evals_out) std::copy(ev.begin(), ev.end(), evals_out);
    return sw;
}

// Eq. 3: Hf = U Delta I_f V^{t*}; with H = U Delta V^{t*} this is Hf = (H V) I_f V^{t*}, written out in
// that order: P = H V (Eq. 6, all k), components outside [k_lo,k_hi] dropped, Hf_t(p) = sum_k P_k(p) conj(V_{t,k}).
extern "C" int oracle_svd_filter(const double* H_, long long n_pix, int T, const double* V_, int k_lo, int k_hi, double* Hf_) {
    if (!H_ || !V_ || !Hf_ || T < 1 || n_pix < 0 || k_lo < 1 || k_hi > T || k_lo > k_hi) return -1;
    std::vector<double> P((size_t)2 * T * n_pix);
    if (oracle_project(H_, n_pix, T, V_, P.data())) return -1;
    const cd* Pc = reinterpret_cast<const cd*>(P.data());
    const cd* V = reinterpret_cast<const cd*>(V_);
    cd* Hf = reinterpret_cast<cd*>(Hf_);
#pragma omp parallel for schedule(static)
    for (int t = 0; t < T; ++t)
        for (long long p = 0; p < n_pix; ++p) {
            cd acc(0, 0);
            for (int k = k_lo; k <= k_hi; ++k) acc += Pc[(long long)(k - 1) * n_pix + p] * std::conj(V[t * T + (k - 1)]);
            Hf[(long long)t * n_pix + p] = acc;
        }
    return 0;
}

// division of an image by its spatial average.
extern "C" int oracle_normalize(const double* M, long long n_pix, double* out) {
    if (!M || !out || n_pix < 1) return -1;
    long double acc = 0.0L;
    for (long long p = 0; p < n_pix; ++p) acc += M[p];
    const double mean = (double)(acc / (long double)n_pix);
    for (long long p = 0; p < n_pix; ++p) out[p] = (mean != 0.0) ? M[p] / mean : M[p];
    return 0;
}

// Quadrant swap (zero-frequency bin to the centre), written as the index map.
extern "C" int oracle_fftshift(const double* in, int ny, int nx, double* out) {
    if (!in || !out || nx < 1 || ny < 1) return -1;
    for (int j = 0; j < ny; ++j)
        for (int i = 0; i < nx; ++i)
            out[(size_t)((j + ny / 2) % ny) * nx + (size_t)((i + nx / 2) % nx)] = in[(size_t)j * nx + i];
    return 0;
}

extern "C" int oracle_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
