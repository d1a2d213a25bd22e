// covariance.cu -- A3: C = H^{t*} H, C_ts = sum_p conj(H_t(p)) H_s(p)   (Eq. 4; R9)
//
// FP32 FFMA Gram of a tall-skinny matrix (N_p x T, T <= 64).  The Hermitian lower half of C is cut
// into 8x8 complex blocks ("jobs"); one warp owns one job and keeps its 64 complex accumulators in
// registers; the 32 lanes split the pixels of a staged chunk (shared memory, cp.async double
// buffer), so the only reduction is a once-per-CTA shuffle tree.  Each CTA writes one partial;
// a second kernel sums the partials in a FIXED order in FP64 (deterministic, bit-identical runs).
#include "holo_internal.cuh"

#define COV_P 128            // pixels per staged chunk
#define COV_MAXW 10          // jobs (warps) per CTA

__device__ __forceinline__ void cp_async16(void* smem, const void* gmem) {
    unsigned s = (unsigned)__cvta_generic_to_shared(smem);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(s), "l"(gmem));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::); }
template <int N> __device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N)); }

// job index -> (block row bi, block col bj), bj <= bi, row-major over the lower triangle
__device__ __forceinline__ void job_to_blocks(int job, int& bi, int& bj) {
    bi = 0;
    while ((bi + 1) * (bi + 2) / 2 <= job) ++bi;
    bj = job - bi * (bi + 1) / 2;
}

// partials layout: [part][T8][T8] float2 (T8 = T rounded up to 8), only blocks bj <= bi are written
template <int T8>
__global__ void __launch_bounds__(COV_MAXW * 32, 1)
k_cov_partial(const float2* __restrict__ H, float2* __restrict__ partials, long long npix, int T,
              int njobs, int jobs_per_cta) {
    extern __shared__ __align__(16) float2 smem[];          // [2][T8][COV_P]
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int nthreads = blockDim.x;
    const int job = blockIdx.y * jobs_per_cta + warp;
    const bool active = (warp < jobs_per_cta) && (job < njobs);
    int bi = 0, bj = 0;
    if (active) job_to_blocks(job, bi, bj);

    // zero the padding rows t >= T of both buffers once
    for (int i = tid; i < 2 * T8 * COV_P; i += nthreads) {
        int row = (i / COV_P) % T8;
        if (row >= T) smem[i] = make_float2(0.f, 0.f);
    }
    const long long nchunks = npix / COV_P;
    const int vec_per_row = COV_P / 2;                       // 16-byte pieces per row
    auto stage = [&](int buf, long long chunk) {
        float2* dst = smem + (size_t)buf * T8 * COV_P;
        const float2* src = H + chunk * COV_P;
        for (int i = tid; i < T * vec_per_row; i += nthreads) {
            int t = i / vec_per_row, v = i - t * vec_per_row;
            cp_async16(dst + t * COV_P + 2 * v, src + (long long)t * npix + 2 * v);
        }
    };

    float2 acc[8][8];
#pragma unroll
    for (int i = 0; i < 8; ++i)
#pragma unroll
        for (int j = 0; j < 8; ++j) acc[i][j] = make_float2(0.f, 0.f);

    long long chunk = blockIdx.x;
    int buf = 0;
    if (chunk < nchunks) stage(0, chunk);
    cp_async_commit();
    for (; chunk < nchunks; chunk += gridDim.x) {
        long long next = chunk + gridDim.x;
        if (next < nchunks) stage(buf ^ 1, next);
        cp_async_commit();
        cp_async_wait<1>();
        __syncthreads();
        if (active) {
            const float2* A = smem + (size_t)buf * T8 * COV_P + (bi * 8) * COV_P;
            const float2* Bm = smem + (size_t)buf * T8 * COV_P + (bj * 8) * COV_P;
#pragma unroll 2
            for (int pp = 0; pp < COV_P / 32; ++pp) {
                const int p = pp * 32 + lane;
                float2 a[8], b[8];
#pragma unroll
                for (int i = 0; i < 8; ++i) a[i] = A[i * COV_P + p];
#pragma unroll
                for (int j = 0; j < 8; ++j) b[j] = Bm[j * COV_P + p];
#pragma unroll
                for (int i = 0; i < 8; ++i)
#pragma unroll
                    for (int j = 0; j < 8; ++j) {            // acc += conj(a_i) * b_j
                        acc[i][j].x = fmaf(a[i].x, b[j].x, acc[i][j].x);
                        acc[i][j].x = fmaf(a[i].y, b[j].y, acc[i][j].x);
                        acc[i][j].y = fmaf(a[i].x, b[j].y, acc[i][j].y);
                        acc[i][j].y = fmaf(-a[i].y, b[j].x, acc[i][j].y);
                    }
            }
        }
        __syncthreads();
        buf ^= 1;
    }
    cp_async_wait<0>();
    if (active) {
        float2* out = partials + (size_t)blockIdx.x * T8 * T8;
#pragma unroll
        for (int i = 0; i < 8; ++i)
#pragma unroll
            for (int j = 0; j < 8; ++j) {
                float x = acc[i][j].x, y = acc[i][j].y;
#pragma unroll
                for (int o = 16; o >= 1; o >>= 1) {
                    x += __shfl_xor_sync(0xffffffffu, x, o);
                    y += __shfl_xor_sync(0xffffffffu, y, o);
                }
                if (lane == 0) out[(bi * 8 + i) * T8 + (bj * 8 + j)] = make_float2(x, y);
            }
    }
}

// fixed-order FP64 reduction over the partials: one warp per lower-triangle entry, lane l sums parts
// l, l+32, ... in order, then a fixed shuffle tree (deterministic).  Writes the full Hermitian C (both
// triangles), diagonal imaginary parts forced to 0.
__global__ void __launch_bounds__(256) k_cov_reduce(const float2* __restrict__ partials, int nparts, int T, int T8, float2* __restrict__ C) {
    const int w = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
    if (w >= T * T) return;
    const int t = w / T, s = w - t * T;
    if (s > t) return;
    double re = 0.0, im = 0.0;
    const float2* p = partials + t * T8 + s;
    for (int k = lane; k < nparts; k += 32) {
        const float2 v = p[(size_t)k * T8 * T8];
        re += (double)v.x;
        im += (double)v.y;
    }
#pragma unroll
    for (int o = 16; o >= 1; o >>= 1) {
        re += __shfl_xor_sync(0xffffffffu, re, o);
        im += __shfl_xor_sync(0xffffffffu, im, o);
    }
    if (lane == 0) {
        if (s == t) {
            C[t * T + t] = make_float2((float)re, 0.f);
        } else {
            C[t * T + s] = make_float2((float)re, (float)im);
            C[s * T + t] = make_float2((float)re, (float)-im);
        }
    }
}

template <int T8>
static int launch_cov_t(holo_ctx* c, const float2* H, float2* C, cudaStream_t st) {
    const int nb = T8 / 8, njobs = nb * (nb + 1) / 2;
    const int jobs_per_cta = njobs < COV_MAXW ? njobs : (njobs == 36 ? 9 : COV_MAXW);
    const int gy = (njobs + jobs_per_cta - 1) / jobs_per_cta;
    const size_t smem = (size_t)2 * T8 * COV_P * sizeof(float2);
    auto kern = k_cov_partial<T8>;
    static bool attr = false;
    if (!attr) {
        HOLO_CUDA_OK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        attr = true;
    }
    long long nchunks = c->npix / COV_P;
    int gx = c->tune[HOLO_TUNE_COV_GRIDX];
    if (gx > c->cov_parts_cap) gx = c->cov_parts_cap;
    if ((long long)gx > nchunks) gx = (int)nchunks;
    {
        HoloProf prof(c, HOLO_K_COV_PARTIAL, st);
        kern<<<dim3(gx, gy), jobs_per_cta * 32, smem, st>>>(H, c->cov_partials, c->npix, c->T, njobs, jobs_per_cta);
    }
    HOLO_CUDA_OK(cudaGetLastError());
    int n = c->T * c->T;
    HoloProf prof(c, HOLO_K_COV_REDUCE, st);
    k_cov_reduce<<<(n * 32 + 255) / 256, 256, 0, st>>>(c->cov_partials, gx, c->T, T8, C);
    HOLO_CUDA_OK(cudaGetLastError());
    return HOLO_OK;
}

int holo_launch_covariance(holo_ctx* c, const float2* H, float2* C, cudaStream_t st) {
    const int T8 = (c->T + 7) / 8 * 8;
    switch (T8) {
        case 8:  return launch_cov_t<8>(c, H, C, st);
        case 16: return launch_cov_t<16>(c, H, C, st);
        case 24: return launch_cov_t<24>(c, H, C, st);
        case 32: return launch_cov_t<32>(c, H, C, st);
        case 40: return launch_cov_t<40>(c, H, C, st);
        case 48: return launch_cov_t<48>(c, H, C, st);
        case 56: return launch_cov_t<56>(c, H, C, st);
        case 64: return launch_cov_t<64>(c, H, C, st);
    }
    holo_set_error("T out of range");
    return HOLO_ERR_ARG;
}
