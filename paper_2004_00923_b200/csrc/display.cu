// display.cu -- the post-processing the paper applies to its images and its SVD-filter form of the clutter rejection:
//   holo_normalize : M <- M / <M>, the division by the spatial average of PAPER.md:86 ("image normalization by their
//                    respective average value is crucial")
//   holo_fftshift  : quadrant swap of an image in FFT-bin order (zero frequency to the centre; R6)
//   holo_svd_filter: H_f = U Delta I_f V^{t*} = H V I_f V^{t*}   (Eq. 3)
// Product code (CUDA, sm_100a); nothing here is shared with oracle/.
#include "holo_internal.cuh"

namespace {

constexpr int NORM_THREADS = 256;

// fixed partition, fixed tree: CTA b sums its contiguous slice in FP64 (thread-strided partial sums, then a shared-memory
// tree) -> partial[b].  Bit-reproducible for a given (npix, grid).
__global__ void __launch_bounds__(NORM_THREADS) k_image_partial_sums(const float* __restrict__ M, long long npix, double* __restrict__ partial) {
    __shared__ double sh[NORM_THREADS];
    const long long per = (npix + gridDim.x - 1) / gridDim.x;
    const long long p0 = (long long)blockIdx.x * per;
    const long long p1 = p0 + per < npix ? p0 + per : npix;
    double acc = 0.0;
    for (long long p = p0 + threadIdx.x; p < p1; p += NORM_THREADS) acc += (double)M[p];
    sh[threadIdx.x] = acc;
    __syncthreads();
    for (int s = NORM_THREADS / 2; s > 0; s >>= 1) {
        if ((int)threadIdx.x < s) sh[threadIdx.x] += sh[threadIdx.x + s];
        __syncthreads();
    }
    if (threadIdx.x == 0) partial[blockIdx.x] = sh[0];
}

// every CTA adds the partials up in the same fixed order (nparts is a few hundred) and scales its slice
__global__ void __launch_bounds__(NORM_THREADS) k_image_scale(float* __restrict__ M, long long npix, const double* __restrict__ partial, int nparts) {
    __shared__ float s_scale;
    if (threadIdx.x == 0) {
        double tot = 0.0;
        for (int i = 0; i < nparts; ++i) tot += partial[i];
        const double mean = tot / (double)npix;
        s_scale = mean != 0.0 ? (float)(1.0 / mean) : 1.f;      // a zero image stays zero
    }
    __syncthreads();
    const float sc = s_scale;
    for (long long p = (long long)blockIdx.x * NORM_THREADS + threadIdx.x; p < npix; p += (long long)gridDim.x * NORM_THREADS) M[p] *= sc;
}

__global__ void __launch_bounds__(256) k_fftshift(const float* __restrict__ in, float* __restrict__ out, int nx, int ny) {
    const long long npix = (long long)nx * ny;
    for (long long p = (long long)blockIdx.x * 256 + threadIdx.x; p < npix; p += (long long)gridDim.x * 256) {
        const int j = (int)(p / nx), i = (int)(p - (long long)j * nx);
        const int js = (j + ny / 2) % ny, is = (i + nx / 2) % nx;
        out[(long long)js * nx + is] = in[p];
    }
}

// F = V I_f V^{t*}:  F[s][t] = sum_{k in [k_lo,k_hi]} V_{s,k} conj(V_{t,k})   (T x T, one small CTA)
__global__ void k_filter_matrix(const float2* __restrict__ V, int T, int k_lo, int k_hi, float2* __restrict__ F) {
    for (int e = threadIdx.x; e < T * T; e += blockDim.x) {
        const int s = e / T, t = e - s * T;
        float2 acc = make_float2(0.f, 0.f);
        for (int k = k_lo - 1; k <= k_hi - 1; ++k) {
            const float2 a = V[s * T + k], b = V[t * T + k];
            acc.x += a.x * b.x + a.y * b.y;               // a conj(b)
            acc.y += a.y * b.x - a.x * b.y;
        }
        F[e] = acc;
    }
}

// Hf_t(p) = sum_s H_s(p) F[s][t]; one pixel per thread, its T holograms in registers, F broadcast from shared memory.
// In place (Hf == H) is allowed: a thread reads all T values of its pixel before it writes any.
template <int TMAX>
__global__ void __launch_bounds__(128) k_svd_filter(const float2* __restrict__ H, const float2* __restrict__ F, float2* __restrict__ Hf,
                                                    long long npix, int T) {
    __shared__ float2 Fs[TMAX * TMAX];                    // [t][s] (transposed: the inner loop walks s)
    for (int e = threadIdx.x; e < TMAX * TMAX; e += blockDim.x) {
        const int t = e / TMAX, s = e - t * TMAX;
        Fs[e] = (t < T && s < T) ? F[s * T + t] : make_float2(0.f, 0.f);
    }
    __syncthreads();
    const long long p = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= npix) return;
    float2 h[TMAX];
#pragma unroll
    for (int s = 0; s < TMAX; ++s) h[s] = s < T ? __ldg(H + (long long)s * npix + p) : make_float2(0.f, 0.f);
#pragma unroll 1
    for (int t = 0; t < T; ++t) {
        const float2* f = Fs + t * TMAX;
        float2 acc = make_float2(0.f, 0.f);
#pragma unroll
        for (int s = 0; s < TMAX; ++s) {
            const float2 w = f[s];
            acc.x = fmaf(h[s].x, w.x, fmaf(-h[s].y, w.y, acc.x));
            acc.y = fmaf(h[s].x, w.y, fmaf(h[s].y, w.x, acc.y));
        }
        Hf[(long long)t * npix + p] = acc;
    }
}

}  // namespace

int holo_launch_normalize(holo_ctx* c, float* image, cudaStream_t st) {
    const int nparts = 2 * c->num_sms < HOLO_NORM_PARTS ? 2 * c->num_sms : HOLO_NORM_PARTS;
    k_image_partial_sums<<<nparts, NORM_THREADS, 0, st>>>(image, c->npix, c->norm_partials);
    HOLO_CUDA_OK(cudaGetLastError());
    k_image_scale<<<4 * c->num_sms, NORM_THREADS, 0, st>>>(image, c->npix, c->norm_partials, nparts);
    HOLO_CUDA_OK(cudaGetLastError());
    return HOLO_OK;
}

int holo_launch_fftshift(holo_ctx* c, const float* in, float* out, cudaStream_t st) {
    k_fftshift<<<4 * c->num_sms, 256, 0, st>>>(in, out, c->nx, c->ny);
    HOLO_CUDA_OK(cudaGetLastError());
    return HOLO_OK;
}

int holo_launch_svd_filter(holo_ctx* c, const float2* H, const float2* V, int k_lo, int k_hi, float2* Hf, cudaStream_t st) {
    const int T = c->T;
    k_filter_matrix<<<1, 256, 0, st>>>(V, T, k_lo, k_hi, c->Fmat);
    HOLO_CUDA_OK(cudaGetLastError());
    const int threads = 128;
    const int grid = (int)((c->npix + threads - 1) / threads);
    if (T <= 8) k_svd_filter<8><<<grid, threads, 0, st>>>(H, c->Fmat, Hf, c->npix, T);
    else if (T <= 16) k_svd_filter<16><<<grid, threads, 0, st>>>(H, c->Fmat, Hf, c->npix, T);
    else if (T <= 32) k_svd_filter<32><<<grid, threads, 0, st>>>(H, c->Fmat, Hf, c->npix, T);
    else k_svd_filter<64><<<grid, threads, 0, st>>>(H, c->Fmat, Hf, c->npix, T);
    HOLO_CUDA_OK(cudaGetLastError());
    return HOLO_OK;
}
