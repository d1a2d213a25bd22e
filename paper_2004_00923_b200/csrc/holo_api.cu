// holo_api.cu -- the C ABI declared in include/holo.h: handle, workspace, argument checks, chaining.
// Every compute step runs in the kernels of fresnel.cu / covariance.cu / eig.cu / project.cu.
#include "holo_internal.cuh"
#include <math.h>
#include <stdarg.h>
#include <string.h>
#include <mutex>
#include <new>
#include <vector>

static thread_local char g_err[512] = "";
int holo_pdl_enabled = 1;

void holo_set_error(const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
}

extern "C" const char* holo_last_error(void) { return g_err; }
extern "C" int holo_version(void) { return 200; }   // 0.2.0

static bool is_pow2(int n) { return n > 0 && (n & (n - 1)) == 0; }

// ---- per-(function, device) caches: the opt-in to > 48 KB dynamic shared memory and the occupancy of a kernel are
// properties of the pair, not of the process (a second handle on another GPU must set them again)
namespace {
struct FuncDevEntry { const void* func; int device; size_t smem; int threads; int occ; };
std::mutex g_fd_mutex;
std::vector<FuncDevEntry> g_fd_attr, g_fd_occ;
}

int holo_ensure_smem_attr(const void* func, int device, size_t bytes) {
    std::lock_guard<std::mutex> lock(g_fd_mutex);
    for (const FuncDevEntry& e : g_fd_attr)
        if (e.func == func && e.device == device && e.smem >= bytes) return HOLO_OK;
    if (bytes > 48 * 1024) HOLO_CUDA_OK(cudaFuncSetAttribute(func, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes));
    g_fd_attr.push_back(FuncDevEntry{func, device, bytes, 0, 0});
    return HOLO_OK;
}

int holo_cached_occupancy(const void* func, int device, int threads, size_t smem, int* blocks_per_sm) {
    {
        std::lock_guard<std::mutex> lock(g_fd_mutex);
        for (const FuncDevEntry& e : g_fd_occ)
            if (e.func == func && e.device == device && e.smem == smem && e.threads == threads) { *blocks_per_sm = e.occ; return HOLO_OK; }
    }
    { const int rc = holo_ensure_smem_attr(func, device, smem); if (rc) return rc; }
    int occ = 0;
    HOLO_CUDA_OK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, func, threads, smem));
    if (occ < 1) { holo_set_error("kernel does not fit on an SM (%d threads, %zu bytes of shared memory)", threads, smem); return HOLO_ERR_CUDA; }
    std::lock_guard<std::mutex> lock(g_fd_mutex);
    g_fd_occ.push_back(FuncDevEntry{func, device, smem, threads, occ});
    *blocks_per_sm = occ;
    return HOLO_OK;
}

static int build_chirp(float2** dst, int n, double lambda_m, double pitch_m, double z_m, double scale) {
    // q_x[i] = exp(+i pi x_i^2/(lambda z)), x_i = (i - n/2) pitch; evaluated in double with the phase
    // reduced mod 2 (in units of pi) BEFORE the trigonometric call (the phase reaches 1e4 rad).
    std::vector<float2> h(n);
    const double PI = 3.14159265358979323846264338327950288;
    const double a = pitch_m * pitch_m / (lambda_m * z_m);      // phase / pi per unit offset^2
    for (int i = 0; i < n; ++i) {
        const double o = (double)(i - n / 2);
        double u = fmod(o * o * a, 2.0);
        h[i] = make_float2((float)(scale * cos(PI * u)), (float)(scale * sin(PI * u)));
    }
    HOLO_CUDA_OK(cudaMalloc(dst, n * sizeof(float2)));
    HOLO_CUDA_OK(cudaMemcpy(*dst, h.data(), n * sizeof(float2), cudaMemcpyHostToDevice));
    return HOLO_OK;
}

static void free_ctx(holo_ctx* c) {
    if (!c) return;
    cudaFree(c->qx); cudaFree(c->qy); cudaFree(c->qxs); cudaFree(c->Wdft); cudaFree(c->Fmat); cudaFree(c->norm_partials);
    holo_fft_plan_free(&c->px); holo_fft_plan_free(&c->py);
    cudaFree(c->sum); cudaFree(c->scratch); cudaFree(c->H); cudaFree(c->rowout); cudaFree(c->cov_partials);
    cudaFree(c->C); cudaFree(c->evals); cudaFree(c->V); cudaFree(c->status);
    if (c->noconv_host) cudaFreeHost(c->noconv_host);
    cudaFree(c->counters); cudaFree(c->gram_X); cudaFree(c->gram_Xp);
    cudaFree(c->defl_img); cudaFree(c->defl_coef); cudaFree(c->energy_parts); cudaFree(c->sum1); cudaFree(c->eig_img);
    if (c->prof_ev) {
        for (int i = 0; i < 2 * HOLO_PROF_CAP; ++i) cudaEventDestroy(c->prof_ev[i]);
        delete[] c->prof_ev;
        delete[] c->prof_cls;
    }
    cudaFree(c->Cd); cudaFree(c->ring); cudaFree(c->Gs);
    cudaFree(c->H1); cudaFree(c->C1); cudaFree(c->evals1); cudaFree(c->V1); cudaFree(c->status1);
    if (c->side) {
        cudaStreamDestroy(c->side);
        for (int i = 0; i < 2; ++i) { cudaEventDestroy(c->ev_cov[i]); cudaEventDestroy(c->ev_eig[i]); cudaEventDestroy(c->ev_proj[i]); }
    }
    if (c->copy) {
        cudaStreamDestroy(c->copy);
        for (int i = 0; i < 2; ++i) { cudaFree(c->fstage[i]); cudaFree(c->istage[i]); cudaEventDestroy(c->ev_h2d[i]); cudaEventDestroy(c->ev_free[i]); }
        if (c->fstage[2]) { cudaFree(c->fstage[2]); cudaEventDestroy(c->ev_h2d[2]); cudaEventDestroy(c->ev_free[2]); }
    }
    if (c->frames_stage) cudaFree(c->frames_stage);
    if (c->image_stage) cudaFree(c->image_stage);
    delete c;
}

static int create_impl(holo_ctx* c) {
    HOLO_CUDA_OK(cudaGetDevice(&c->device));
    cudaDeviceProp prop;
    HOLO_CUDA_OK(cudaGetDeviceProperties(&prop, c->device));
    if (prop.major < 10) { holo_set_error("libholo_b200 needs an sm_100a device (found sm_%d%d)", prop.major, prop.minor); return HOLO_ERR_CUDA; }
    c->num_sms = prop.multiProcessorCount;
    const int T = c->T;
    const long long np = c->npix;
    int rc;
    if ((rc = build_chirp(&c->qx, c->nx, c->lambda_m, c->pitch_m, c->z_m, 1.0))) return rc;
    if ((rc = build_chirp(&c->qy, c->ny, c->lambda_m, c->pitch_m, c->z_m, 1.0))) return rc;
    if ((rc = build_chirp(&c->qxs, c->nx, c->lambda_m, c->pitch_m, c->z_m, 1.0 / (double)c->T))) return rc;
    if ((rc = holo_fft_plan_init(&c->px, c->nx))) return rc;
    if ((rc = holo_fft_plan_init(&c->py, c->ny))) return rc;
    {   // Eq. 8: w_mn = exp(-2 i pi (m-1)(n-1)/T)/sqrt(T)
        std::vector<float2> W((size_t)T * T);
        const double PI = 3.14159265358979323846264338327950288;
        for (int m = 0; m < T; ++m)
            for (int n = 0; n < T; ++n) {
                const double ang = -2.0 * PI * (double)((m * n) % T) / (double)T;
                W[(size_t)m * T + n] = make_float2((float)(cos(ang) / sqrt((double)T)), (float)(sin(ang) / sqrt((double)T)));
            }
        HOLO_CUDA_OK(cudaMalloc(&c->Wdft, W.size() * sizeof(float2)));
        HOLO_CUDA_OK(cudaMemcpy(c->Wdft, W.data(), W.size() * sizeof(float2), cudaMemcpyHostToDevice));
    }
    // tuning defaults
    long long grp = (48ll << 20) / (8 * np);                 // keep the FFT intermediate <= 48 MiB (L2-resident)
    if (grp < 3) grp = 3;                                    // the fused kernel needs a ring of >= 2 frames; 3 measured 11 % faster at 2048^2
    if (grp > T) grp = T;
    c->tune[HOLO_TUNE_FFT_GROUP] = (int)grp;
    c->tune[HOLO_TUNE_COV_GRIDX] = c->num_sms;
    c->tune[HOLO_TUNE_PROJ_COMPLEMENT] = 1;
    c->tune[HOLO_TUNE_FFT_PERSISTENT] = 1;
    c->tune[HOLO_TUNE_PROJ_TMA] = 1;
    c->tune[HOLO_TUNE_COV_REAL] = 1;
    c->tune[HOLO_TUNE_PUSH_PIPE] = 1;
    c->tune[HOLO_TUNE_PUSH_INCR] = 1;
    // 40 of 148 SMs: measured optimum at 1024^2 x 32 (354 -> 320 us per stack); at T = 64 the projection is too slow
    // per SM (64 holograms in registers) and the split loses (3.87 -> 4.30 ms), so it is off there
    c->tune[HOLO_TUNE_SPLIT_SMS] = T <= 32 ? (c->num_sms * 27 + 50) / 100 : 0;
    c->tune[HOLO_TUNE_EIG_MAX_SWEEPS] = 30;
    // real covariance on the tensor cores (TF32, inputs rounded to nearest, accumulators added to FP64 every 4 stages = 512
    // products): measured 584 vs 919 us at 2048^2 x 64 with 2e-6 on the eigenvalues; at T <= 32 the gain is 12 % (75 vs 85 us)
    // and the FP32 kernel stays the default (profiles/r02_tf32_gram.md)
    // (the rounding noise of single-pass TF32 averages out as 1 / sqrt(pixels): below 2^20 pixels the split form is used)
    // tensor-core covariance: at T > 32 (the FP32 kernel is ALU bound there; 3 x TF32 below 2^20 pixels, where the rounding noise
    // of a single pass has too few products to average over), and at T = 32 from 2^18 pixels in a single pass (measured against
    // the oracle: C 3.3e-6 / eigenvalues 2.4e-6 / image 2.5e-7 at 512^2, 2.7e-6 / 2.5e-6 / 2.6e-7 at 1024^2; the FP32 kernel:
    // 2e-7 / 2e-7 / 2.1e-7): 300 vs 321 us per stack at 1024^2, 99 vs 108 us at 512^2
    c->tune[HOLO_TUNE_COV_TF32] = (np % 256 != 0) ? 0 : T > 32 ? (np >= (1ll << 20) ? 1 : 3) : (T == 32 && np >= (1ll << 18)) ? 1 : 0;
    c->tune[HOLO_TUNE_COV_TF32_DRAIN] = 4;
    c->tune[HOLO_TUNE_PROJ_TC] = 1;
    c->tune[HOLO_TUNE_COLS2048] = 1;
    c->tune[HOLO_TUNE_TILED_G] = 8;
    c->tune[HOLO_TUNE_COV_TF32_TMA] = 1;
    c->tune[HOLO_TUNE_PACKED1024] = 1;
    c->tune[HOLO_TUNE_PDL] = holo_pdl_enabled;
    c->tune[HOLO_TUNE_ROWS2] = 1;                // packed two-frame row pass of mode 3 (1024^2, even T): 79 vs 84 us
    c->scratch_frames = (int)grp;
    c->cov_parts_cap = 4 * c->num_sms;
    const int T8 = (T + 7) / 8 * 8;
    HOLO_CUDA_OK(cudaMalloc(&c->sum, np * sizeof(uint32_t)));
    HOLO_CUDA_OK(cudaMalloc(&c->scratch, (size_t)c->scratch_frames * np * sizeof(float2)));
    HOLO_CUDA_OK(cudaMalloc(&c->H, (size_t)T * np * sizeof(float2)));
    if ((c->nx == 2048 && c->ny == 2048) || (c->nx == 1024 && c->ny == 1024 && T % 2 == 0 && T >= 16))
        HOLO_CUDA_OK(cudaMalloc(&c->rowout, (size_t)T * np * sizeof(float2)));
    HOLO_CUDA_OK(cudaMalloc(&c->cov_partials, (size_t)c->cov_parts_cap * T8 * T8 * sizeof(float2)));
    HOLO_CUDA_OK(cudaMalloc(&c->C, (size_t)T * T * sizeof(float2)));
    HOLO_CUDA_OK(cudaMalloc(&c->evals, T * sizeof(float)));
    HOLO_CUDA_OK(cudaMalloc(&c->V, (size_t)T * T * sizeof(float2)));
    HOLO_CUDA_OK(cudaMalloc(&c->status, 8 * sizeof(int32_t)));
    HOLO_CUDA_OK(cudaMalloc(&c->counters, 1024 * sizeof(unsigned int)));
    HOLO_CUDA_OK(cudaMalloc(&c->gram_X, 128 * 128 * sizeof(unsigned long long)));
    {
        const size_t Ng = T <= 32 ? 64 : 128;
        HOLO_CUDA_OK(cudaMalloc(&c->gram_Xp, Ng * (Ng + 1) / 2 * (size_t)(3 * c->num_sms) * sizeof(unsigned long long)));
    }
    HOLO_CUDA_OK(cudaMalloc(&c->Fmat, (size_t)T * T * sizeof(float2)));
    HOLO_CUDA_OK(cudaMalloc(&c->norm_partials, HOLO_NORM_PARTS * sizeof(double)));
    c->mode = 1;
    HOLO_CUDA_OK(cudaMemset(c->status, 0, 8 * sizeof(int32_t)));
    HOLO_CUDA_OK(cudaMemset(c->counters, 0, 1024 * sizeof(unsigned int)));
    HOLO_CUDA_OK(cudaMemset(c->cov_partials, 0, (size_t)c->cov_parts_cap * T8 * T8 * sizeof(float2)));
    HOLO_CUDA_OK(cudaHostAlloc(&c->noconv_host, sizeof(int32_t), cudaHostAllocMapped));
    *c->noconv_host = 0;
    HOLO_CUDA_OK(cudaHostGetDevicePointer((void**)&c->noconv_dev, c->noconv_host, 0));
    HOLO_CUDA_OK(cudaDeviceSynchronize());
    return HOLO_OK;
}

extern "C" holo_ctx* holo_create(int nx, int ny, int T, double lambda_m, double pitch_m, double z_m,
                                 int k_lo, int k_hi) {
    if (!is_pow2(nx) || !is_pow2(ny) || nx < 16 || ny < 16 || nx > 4096 || ny > 4096) {
        holo_set_error("nx, ny must be powers of two in [16, 4096] (got %d x %d)", nx, ny);
        return nullptr;
    }
    if (T < 2 || T > HOLO_MAX_T) { holo_set_error("T must be in [2, %d] (got %d)", HOLO_MAX_T, T); return nullptr; }
    if (!(lambda_m > 0) || !(pitch_m > 0) || !(z_m > 0) || !isfinite(lambda_m) || !isfinite(pitch_m) || !isfinite(z_m)) {
        holo_set_error("lambda, pitch, z must be finite and > 0");
        return nullptr;
    }
    if (k_lo < 1 || k_hi > T || k_lo > k_hi) { holo_set_error("need 1 <= k_lo <= k_hi <= T (got %d, %d)", k_lo, k_hi); return nullptr; }
    holo_ctx* c = new (std::nothrow) holo_ctx();
    if (!c) { holo_set_error("out of host memory"); return nullptr; }
    memset(c, 0, sizeof(*c));
    c->nx = nx; c->ny = ny; c->T = T; c->npix = (long long)nx * ny;
    c->lambda_m = lambda_m; c->pitch_m = pitch_m; c->z_m = z_m;
    c->k_lo = k_lo; c->k_hi = k_hi;
    if (create_impl(c) != HOLO_OK) { free_ctx(c); return nullptr; }
    return c;
}

extern "C" void holo_destroy(holo_ctx* c) {
    if (!c) return;
    cudaDeviceSynchronize();
    free_ctx(c);
}

// Every entry point: the handle's device must be current (its streams, events and per-device kernel attributes belong
// to it), and a Jacobi solve of an EARLIER call that hit the sweep cap is reported once, before anything is enqueued
// (the eigensolver sets a mapped host word; no synchronisation here -- SURVEY.md 8(b)).
static int enter(holo_ctx* c, bool report_noconv = true) {
    if (!c) { holo_set_error("NULL handle"); return HOLO_ERR_ARG; }
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev != c->device) {
        holo_set_error("the handle was created on device %d but device %d is current", c->device, dev);
        return HOLO_ERR_STATE;
    }
    if (report_noconv && c->noconv_host && *(volatile int32_t*)c->noconv_host) {
        *(volatile int32_t*)c->noconv_host = 0;
        holo_set_error("the Jacobi eigensolver of an earlier call hit the sweep cap (see holo_status)");
        return HOLO_ERR_NOCONV;
    }
    return HOLO_OK;
}
#define CHECK_CTX(c) do { const int _rc = enter(c); if (_rc) return _rc; } while (0)
#define CHECK_CTX_QUIET(c) do { const int _rc = enter(c, false); if (_rc) return _rc; } while (0)
#define CHECK_PTR(p, name) do { if (!(p)) { holo_set_error("NULL pointer: %s", name); return HOLO_ERR_ARG; } } while (0)

extern "C" int holo_fresnel(holo_ctx* c, const uint16_t* frames_dev, void* H_dev, holo_stream stream) {
    CHECK_CTX(c); CHECK_PTR(frames_dev, "frames_dev"); CHECK_PTR(H_dev, "H_dev");
    if (((uintptr_t)frames_dev & 15) || ((uintptr_t)H_dev & 15)) { holo_set_error("frames_dev/H_dev must be 16-byte aligned"); return HOLO_ERR_ARG; }
    return holo_launch_fresnel(c, frames_dev, (float2*)H_dev, (cudaStream_t)stream);
}

extern "C" int holo_covariance(holo_ctx* c, const void* H_dev, void* C_dev, holo_stream stream) {
    CHECK_CTX(c); CHECK_PTR(H_dev, "H_dev"); CHECK_PTR(C_dev, "C_dev");
    if ((uintptr_t)H_dev & 15) { holo_set_error("H_dev must be 16-byte aligned"); return HOLO_ERR_ARG; }
    return holo_launch_covariance(c, (const float2*)H_dev, (float2*)C_dev, (cudaStream_t)stream);
}

extern "C" int holo_eig(holo_ctx* c, const void* C_dev, float* evals_dev, void* V_dev, holo_stream stream) {
    CHECK_CTX(c); CHECK_PTR(C_dev, "C_dev"); CHECK_PTR(evals_dev, "evals_dev"); CHECK_PTR(V_dev, "V_dev");
    return holo_launch_eig(c, (const float2*)C_dev, evals_dev, (float2*)V_dev, (cudaStream_t)stream);
}

extern "C" int holo_project(holo_ctx* c, const void* H_dev, const void* V_dev, float* image_dev, holo_stream stream) {
    CHECK_CTX(c); CHECK_PTR(H_dev, "H_dev"); CHECK_PTR(V_dev, "V_dev"); CHECK_PTR(image_dev, "image_dev");
    if (((uintptr_t)H_dev & 15) || ((uintptr_t)image_dev & 7)) { holo_set_error("H_dev must be 16-byte and image_dev 8-byte aligned"); return HOLO_ERR_ARG; }
    return holo_launch_project(c, (const float2*)H_dev, (const float2*)V_dev, c->k_lo, c->k_hi,
                               c->assume_unitary, image_dev, (cudaStream_t)stream);
}

extern "C" int holo_fourier_demod(holo_ctx* c, const void* H_dev, int n1, int n2, float* image_dev, holo_stream stream) {
    CHECK_CTX(c); CHECK_PTR(H_dev, "H_dev"); CHECK_PTR(image_dev, "image_dev");
    if (n1 < 1 || n2 > c->T || n1 > n2) { holo_set_error("need 1 <= n1 <= n2 <= T"); return HOLO_ERR_ARG; }
    if (((uintptr_t)H_dev & 15) || ((uintptr_t)image_dev & 7)) { holo_set_error("H_dev must be 16-byte and image_dev 8-byte aligned"); return HOLO_ERR_ARG; }
    return holo_launch_project(c, (const float2*)H_dev, c->Wdft, n1, n2, /*W is unitary*/ 1, image_dev, (cudaStream_t)stream);
}

extern "C" int holo_svd_filter(holo_ctx* c, const void* H_dev, const void* V_dev, void* Hf_dev, holo_stream stream) {
    CHECK_CTX(c); CHECK_PTR(H_dev, "H_dev"); CHECK_PTR(V_dev, "V_dev"); CHECK_PTR(Hf_dev, "Hf_dev");
    if (((uintptr_t)H_dev & 7) || ((uintptr_t)Hf_dev & 7)) { holo_set_error("H_dev and Hf_dev must be 8-byte aligned"); return HOLO_ERR_ARG; }
    return holo_launch_svd_filter(c, (const float2*)H_dev, (const float2*)V_dev, c->k_lo, c->k_hi, (float2*)Hf_dev, (cudaStream_t)stream);
}

extern "C" int holo_normalize(holo_ctx* c, float* image_dev, holo_stream stream) {
    CHECK_CTX(c); CHECK_PTR(image_dev, "image_dev");
    return holo_launch_normalize(c, image_dev, (cudaStream_t)stream);
}

extern "C" int holo_fftshift(holo_ctx* c, const float* in_dev, float* out_dev, holo_stream stream) {
    CHECK_CTX(c); CHECK_PTR(in_dev, "in_dev"); CHECK_PTR(out_dev, "out_dev");
    if (in_dev == out_dev) { holo_set_error("holo_fftshift works out of place: in_dev == out_dev"); return HOLO_ERR_ARG; }
    return holo_launch_fftshift(c, in_dev, out_dev, (cudaStream_t)stream);
}

static int project_pending(holo_ctx* c, cudaStream_t st);
static int energy_pending(holo_ctx* c, cudaStream_t st);
static int join_side(holo_ctx* c, cudaStream_t st, int slot);

extern "C" int holo_process(holo_ctx* c, const uint16_t* frames_dev, float* image_dev, holo_stream stream) {
    CHECK_CTX(c); CHECK_PTR(frames_dev, "frames_dev"); CHECK_PTR(image_dev, "image_dev");
    if (((uintptr_t)frames_dev & 15) || ((uintptr_t)image_dev & 7)) { holo_set_error("frames_dev must be 16-byte and image_dev 8-byte aligned"); return HOLO_ERR_ARG; }
    cudaStream_t st = (cudaStream_t)stream;
    int rc;
    if ((rc = join_side(c, st, -1))) return rc;
    if ((rc = project_pending(c, st))) return rc;          // a holo_submit still owes its image: deliver it first
    if ((rc = energy_pending(c, st))) return rc;
    c->nsubmit = 0;                                        // the next holo_submit starts again with slot 0
    c->push_ready = 0;                                     // ... and a holo_push sequence has to start over
    if (c->mode == 3) {
        // mode 2's covariance and eigenvectors, then the image straight from the raw frames: rejected components removed in
        // the raw domain, row pass, column pass reduced to sum_t |.|^2 -- no hologram stack, no projection kernel
        if ((rc = holo_launch_sum_gram(c, frames_dev, c->C, st))) return rc;
        if ((rc = holo_launch_eig(c, c->C, c->evals, c->V, st, true))) return rc;
        return holo_launch_energy_image(c, frames_dev, c->V, c->k_lo, c->k_hi, image_dev, st);
    }
    if (c->mode == 2) {
        // covariance from the raw frames (exact integer Gram on the tensor cores, fused with the temporal sum): C and V are
        // known BEFORE the holograms exist, and the hologram stack is read once (projection) instead of twice
        if ((rc = holo_launch_sum_gram(c, frames_dev, c->C, st))) return rc;
        if ((rc = holo_launch_eig(c, c->C, c->evals, c->V, st, true))) return rc;
        if ((rc = holo_launch_fresnel(c, frames_dev, c->H, st, /*with_sum=*/false, -1, /*counters_zeroed=*/true))) return rc;
        return holo_launch_project(c, c->H, c->V, c->k_lo, c->k_hi, c->tune[HOLO_TUNE_PROJ_COMPLEMENT], image_dev, st);
    }
    if ((rc = holo_launch_fresnel(c, frames_dev, c->H, st))) return rc;
    if ((rc = holo_launch_covariance(c, c->H, c->C, st, /*real_only=*/true))) return rc;
    if ((rc = holo_launch_eig(c, c->C, c->evals, c->V, st, c->tune[HOLO_TUNE_COV_REAL] != 0))) return rc;
    return holo_launch_project(c, c->H, c->V, c->k_lo, c->k_hi, c->tune[HOLO_TUNE_PROJ_COMPLEMENT], image_dev, st);
}

extern "C" int holo_raw_covariance(holo_ctx* c, const uint16_t* frames_dev, void* C_dev, holo_stream stream) {
    CHECK_CTX(c); CHECK_PTR(frames_dev, "frames_dev"); CHECK_PTR(C_dev, "C_dev");
    if ((uintptr_t)frames_dev & 15) { holo_set_error("frames_dev must be 16-byte aligned"); return HOLO_ERR_ARG; }
    return holo_launch_sum_gram(c, frames_dev, (float2*)C_dev, (cudaStream_t)stream);
}

// mode 3: a window that takes the eigen-basis form needs its image workspace (allocated once, here: never inside a
// compute call)
static int mode3_prepare(holo_ctx* c, int k_lo, int k_hi) {
    if (holo_mode3_eigen_form(c, k_lo, k_hi) && !c->eig_img)
        HOLO_CUDA_OK(cudaMalloc(&c->eig_img, (size_t)c->T * c->npix * sizeof(float)));
    return HOLO_OK;
}

extern "C" int holo_set_mode(holo_ctx* c, int mode) {
    CHECK_CTX_QUIET(c);
    if (mode < 1 || mode > 3) { holo_set_error("mode must be 1 (covariance of the hologram stack), 2 (of the raw frames) or 3 (2 + image without the hologram stack)"); return HOLO_ERR_ARG; }
    if (c->pend_image || c->pend3_image || c->proj_recorded[0] || c->proj_recorded[1]) { holo_set_error("holo_flush the open holo_submit sequence before changing the mode"); return HOLO_ERR_STATE; }
    if (mode == 3) {
        { const int rc3 = mode3_prepare(c, c->k_lo, c->k_hi); if (rc3) return rc3; }
        if (!c->defl_img) {                                  // first use: the mode's own workspace (allocation, may synchronise)
            HOLO_CUDA_OK(cudaMalloc(&c->defl_img, (size_t)4 * c->npix * sizeof(float)));
            HOLO_CUDA_OK(cudaMalloc(&c->defl_coef, (size_t)HOLO_MAX_T * 4 * sizeof(float)));
            HOLO_CUDA_OK(cudaMalloc(&c->energy_parts, (size_t)8 * c->npix * sizeof(float)));
        }
    }
    c->mode = mode;
    return HOLO_OK;
}

// ---- streaming form: software pipeline over consecutive stacks -------------------------------------
// submit(i) enqueues on `stream`:  A0+A1+A2 of stack i  ->  [join eig(i-1)] A5+A6 of stack i-1  ->  A3 of
// stack i  ->  fork: A4 of stack i on the handle's side stream.  The single-CTA eigensolver of stack i thus
// runs under the Fresnel kernels of stack i+1 instead of idling 147 SMs; everything else keeps stream order.
static int submit_init(holo_ctx* c, bool second_stack = true) {
    const size_t T = (size_t)c->T;
    if (second_stack && !c->H1) HOLO_CUDA_OK(cudaMalloc(&c->H1, T * c->npix * sizeof(float2)));
    if (c->side) return HOLO_OK;
    HOLO_CUDA_OK(cudaMalloc(&c->C1, T * T * sizeof(float2)));
    HOLO_CUDA_OK(cudaMalloc(&c->evals1, T * sizeof(float)));
    HOLO_CUDA_OK(cudaMalloc(&c->V1, T * T * sizeof(float2)));
    HOLO_CUDA_OK(cudaMalloc(&c->status1, 8 * sizeof(int32_t)));
    HOLO_CUDA_OK(cudaMemset(c->status1, 0, 8 * sizeof(int32_t)));
    int lo = 0, hi = 0;
    HOLO_CUDA_OK(cudaDeviceGetStreamPriorityRange(&lo, &hi));
    HOLO_CUDA_OK(cudaStreamCreateWithPriority(&c->side, cudaStreamNonBlocking, hi));
    for (int i = 0; i < 2; ++i) {
        HOLO_CUDA_OK(cudaEventCreateWithFlags(&c->ev_cov[i], cudaEventDisableTiming));
        HOLO_CUDA_OK(cudaEventCreateWithFlags(&c->ev_eig[i], cudaEventDisableTiming));
        HOLO_CUDA_OK(cudaEventCreateWithFlags(&c->ev_proj[i], cudaEventDisableTiming));
    }
    return HOLO_OK;
}

// SM-split mode: make `st` wait for the projections that were enqueued on the side stream
static int join_side(holo_ctx* c, cudaStream_t st, int slot /* -1: both */) {
    for (int s = 0; s < 2; ++s)
        if ((slot < 0 || slot == s) && c->proj_recorded[s]) {
            HOLO_CUDA_OK(cudaStreamWaitEvent(st, c->ev_proj[s], 0));
            if (slot < 0) c->proj_recorded[s] = 0;
        }
    return HOLO_OK;
}

static int project_pending(holo_ctx* c, cudaStream_t st) {
    if (!c->pend_image) return HOLO_OK;
    const int s = c->pend_slot;
    HOLO_CUDA_OK(cudaStreamWaitEvent(st, c->ev_eig[s], 0));
    const int rc = holo_launch_project(c, s ? c->H1 : c->H, s ? c->V1 : c->V, c->pend_k_lo, c->pend_k_hi,
                                       c->pend_complement, c->pend_image, st);      // the window of ITS submit call
    c->pend_image = nullptr;
    return rc;
}

// mode 3, streaming form: the stack whose image is still owed (its frames are read again by the energy pass)
static int energy_pending(holo_ctx* c, cudaStream_t st) {
    if (!c->pend3_image) return HOLO_OK;
    const int s = c->pend3_slot;
    HOLO_CUDA_OK(cudaStreamWaitEvent(st, c->ev_eig[s], 0));
    uint32_t* sum_main = c->sum;
    if (s) c->sum = c->sum1;
    const int rc = holo_launch_energy_image(c, c->pend3_frames, s ? c->V1 : c->V, c->pend_k_lo, c->pend_k_hi, c->pend3_image, st);
    c->sum = sum_main;
    c->pend3_image = nullptr; c->pend3_frames = nullptr;
    return rc;
}

extern "C" int holo_submit(holo_ctx* c, const uint16_t* frames_dev, float* image_dev, holo_stream stream) {
    CHECK_CTX(c); CHECK_PTR(frames_dev, "frames_dev"); CHECK_PTR(image_dev, "image_dev");
    if (((uintptr_t)frames_dev & 15) || ((uintptr_t)image_dev & 7)) { holo_set_error("frames_dev must be 16-byte and image_dev 8-byte aligned"); return HOLO_ERR_ARG; }
    cudaStream_t st = (cudaStream_t)stream;
    int rc;
    if (c->mode == 3) {
        // mode 3: everything of a stack needs its eigenvectors first (the rejected components are removed in the raw domain),
        // so the pipeline is: covariance of stack i (tensor cores, from the raw frames) -> fork its eigensolver to the side
        // stream -> image of stack i-1 (deflation images, row pass, column energy) with the eigensolver of stack i under it.
        // frames_dev of stack i is read AGAIN by the next holo_submit / holo_flush: it must stay valid until then.
        if ((rc = submit_init(c, /*second_stack=*/false))) return rc;
        if (!c->sum1) HOLO_CUDA_OK(cudaMalloc(&c->sum1, (size_t)c->npix * sizeof(uint32_t)));
        c->push_ready = 0;
        const int s = (int)(c->nsubmit & 1);
        // (the Gram pass itself stays on the main stream: on the side stream, next to the transforms of stack i-1, it was
        // measured slower, 219 vs 214 us per stack -- its CTAs do not fit beside the row pass and then delay the eigensolver)
        uint32_t* sum_main = c->sum;
        if (s) c->sum = c->sum1;
        rc = holo_launch_sum_gram(c, frames_dev, s ? c->C1 : c->C, st, /*finish=*/false);
        c->sum = sum_main;
        if (rc) return rc;
        HOLO_CUDA_OK(cudaEventRecord(c->ev_cov[s], st));
        HOLO_CUDA_OK(cudaStreamWaitEvent(c->side, c->ev_cov[s], 0));
        if ((rc = holo_launch_gram_finish(c, s ? c->C1 : c->C, c->side))) return rc;     // off the main stream's critical path
        int32_t* status_main = c->status;
        if (s) c->status = c->status1;
        rc = holo_launch_eig(c, s ? c->C1 : c->C, s ? c->evals1 : c->evals, s ? c->V1 : c->V, c->side, true);
        c->status = status_main;
        if (rc) return rc;
        HOLO_CUDA_OK(cudaEventRecord(c->ev_eig[s], c->side));
        if ((rc = energy_pending(c, st))) return rc;              // image of stack i-1
        c->pend3_image = image_dev; c->pend3_frames = frames_dev; c->pend3_slot = s;
        c->pend_k_lo = c->k_lo; c->pend_k_hi = c->k_hi;
        c->nsubmit++;
        return HOLO_OK;
    }
    if (c->mode == 2) {
        // mode 2: the eigensolver runs on the side stream UNDER the Fresnel stage of the same stack (C comes from the raw
        // frames), so the projection follows in stream order and the image is complete when this call's work is done
        if ((rc = submit_init(c, /*second_stack=*/false))) return rc;
        c->push_ready = 0;
        // the Gram finish (260 small CTAs) stays on the main stream; only the single-CTA eigensolver goes to the side stream,
        // and the persistent Fresnel launch leaves one SM to it (otherwise it fills every SM and the eigensolver waits for
        // its end: measured 324 vs 281 us per stack)
        if ((rc = holo_launch_sum_gram(c, frames_dev, c->C, st, /*finish=*/true))) return rc;
        HOLO_CUDA_OK(cudaEventRecord(c->ev_cov[0], st));
        HOLO_CUDA_OK(cudaStreamWaitEvent(c->side, c->ev_cov[0], 0));
        if ((rc = holo_launch_eig(c, c->C, c->evals, c->V, c->side, true))) return rc;
        HOLO_CUDA_OK(cudaEventRecord(c->ev_eig[0], c->side));
        c->fresnel_sm_reserve = 1;
        rc = holo_launch_fresnel(c, frames_dev, c->H, st, /*with_sum=*/false, -1, /*counters_zeroed=*/true);
        c->fresnel_sm_reserve = 0;
        if (rc) return rc;
        HOLO_CUDA_OK(cudaStreamWaitEvent(st, c->ev_eig[0], 0));
        c->nsubmit++;
        return holo_launch_project(c, c->H, c->V, c->k_lo, c->k_hi, c->tune[HOLO_TUNE_PROJ_COMPLEMENT], image_dev, st);
    }
    if ((rc = submit_init(c))) return rc;
    c->push_ready = 0;
    const int s = (int)(c->nsubmit & 1);
    float2* H = s ? c->H1 : c->H;
    float2* C = s ? c->C1 : c->C;
    // the SM split pairs the HBM-bound DEFLATION projection with the ALU-bound covariance; a wide rejection set takes the
    // direct (tensor-core) projection, which needs the whole GPU: stream order then
    const int nS_now = c->k_hi - c->k_lo + 1;
    const bool deflating = c->tune[HOLO_TUNE_PROJ_COMPLEMENT] && 2 * (c->T - nS_now) <= nS_now;
    // The split pays under the FUSED Fresnel kernel (latency bound at 27 % of the HBM peak: the side-stream projection of the
    // previous stack runs beside it for free).  The packed row / column kernels stream at ~80 % of the HBM peak and need whole
    // SMs: a projection beside them only takes bandwidth and SMs away (339 vs 321 us per stack): stream order then.
    const int split = deflating && !holo_fresnel_is_packed(c) ? c->tune[HOLO_TUNE_SPLIT_SMS] : 0;
    if (c->tune[HOLO_TUNE_SPLIT_SMS] > 0) { if ((rc = join_side(c, st, s))) return rc; }      // H / V of slot s are free once the projection of stack i-2 is done
    if ((rc = holo_launch_fresnel(c, frames_dev, H, st))) return rc;
    if ((rc = project_pending(c, st))) return rc;
    c->cov_grid_cap = split > 0 ? c->num_sms - split : 0;
    rc = holo_launch_covariance(c, H, C, st, /*real_only=*/true);
    c->cov_grid_cap = 0;
    if (rc) return rc;
    // (moving the 8 us partial reduction to the side stream as well gains 3 us at 1024^2 x 32 but loses 7 us at
    //  512^2 x 32, where the side stream -- eigensolver + projection -- is the longer chain)
    HOLO_CUDA_OK(cudaEventRecord(c->ev_cov[s], st));
    HOLO_CUDA_OK(cudaStreamWaitEvent(c->side, c->ev_cov[s], 0));
    int32_t* status_main = c->status;
    if (s) c->status = c->status1;
    rc = holo_launch_eig(c, C, s ? c->evals1 : c->evals, s ? c->V1 : c->V, c->side, c->tune[HOLO_TUNE_COV_REAL] != 0);
    c->status = status_main;
    if (rc) return rc;
    HOLO_CUDA_OK(cudaEventRecord(c->ev_eig[s], c->side));
    if (split > 0) {
        // the projection follows the eigensolver on the side stream and runs on `split` SMs next to the covariance
        // of the next stack; the image is complete after the submit after next, or after holo_flush
        c->proj_grid_cap = split;
        rc = holo_launch_project(c, H, s ? c->V1 : c->V, c->k_lo, c->k_hi, c->tune[HOLO_TUNE_PROJ_COMPLEMENT], image_dev, c->side);
        c->proj_grid_cap = 0;
        if (rc) return rc;
        HOLO_CUDA_OK(cudaEventRecord(c->ev_proj[s], c->side));
        c->proj_recorded[s] = 1;
        c->nsubmit++;
        return HOLO_OK;
    }
    c->pend_image = image_dev; c->pend_slot = s; c->nsubmit++;
    c->pend_k_lo = c->k_lo; c->pend_k_hi = c->k_hi; c->pend_complement = c->tune[HOLO_TUNE_PROJ_COMPLEMENT];
    return HOLO_OK;
}

extern "C" int holo_flush(holo_ctx* c, holo_stream stream) {
    CHECK_CTX(c);
    int rc = join_side(c, (cudaStream_t)stream, -1);
    if (rc) return rc;
    if ((rc = energy_pending(c, (cudaStream_t)stream))) return rc;
    return project_pending(c, (cudaStream_t)stream);
}

// ---- sliding window (BASELINE.json configs[3]) ------------------------------------
// The handle's hologram stack is used as a ring of the T most recent frames.  The holograms are taken against a
// FIXED reference image m0 (the temporal mean of the first window; its sum image S0 stays in ctx->sum), G_t =
// F[q (I_t - m0)], so a frame is transformed ONCE and stays valid while the window slides; the window's own mean
// is removed afterwards, exactly (linearity): H_t = G_t - mean_t G.  Covariance: C = J (G^H G) J, centred in FP64
// (k_center_gram); projection: the deflation kernel subtracts the per-pixel mean first.  Row / column order of C
// follows the ring slots, which permutes C, V symmetrically and leaves eigenvalues and M unchanged.
static bool push_ring_possible(const holo_ctx* c) {
    return c->tune[HOLO_TUNE_PUSH_PIPE] && (c->T == 16 || c->T == 32 || c->T == 64) && c->tune[HOLO_TUNE_COV_REAL] && c->tune[HOLO_TUNE_PROJ_TMA];
}

// window of the ring -> ctx->H (contiguous), when a push cannot use the ring (n_new not a multiple of 8, or too large)
static int push_ring_to_flat(holo_ctx* c, cudaStream_t st) {
    int rc;
    if ((rc = join_side(c, st, -1))) return rc;
    const int T = c->T, Rn = c->ring_slots;
    const int first = (Rn - c->ring_a < T) ? Rn - c->ring_a : T;
    HOLO_CUDA_OK(cudaMemcpyAsync(c->H, c->ring + (size_t)c->ring_a * c->npix, (size_t)first * c->npix * sizeof(float2), cudaMemcpyDeviceToDevice, st));
    if (first < T)
        HOLO_CUDA_OK(cudaMemcpyAsync(c->H + (size_t)first * c->npix, c->ring, (size_t)(T - first) * c->npix * sizeof(float2), cudaMemcpyDeviceToDevice, st));
    c->push_ready = 1; c->push_head = 0;
    return HOLO_OK;
}

extern "C" int holo_push(holo_ctx* c, const uint16_t* new_frames_dev, int n_new, float* image_dev, holo_stream stream) {
    CHECK_CTX(c); CHECK_PTR(new_frames_dev, "new_frames_dev"); CHECK_PTR(image_dev, "image_dev");
    if (((uintptr_t)new_frames_dev & 15) || ((uintptr_t)image_dev & 7)) { holo_set_error("new_frames_dev must be 16-byte and image_dev 8-byte aligned"); return HOLO_ERR_ARG; }
    const int T = c->T;
    if (n_new < 1 || n_new > T) { holo_set_error("need 1 <= n_new <= T (got %d)", n_new); return HOLO_ERR_ARG; }
    if (!c->push_ready && n_new != T) { holo_set_error("the first holo_push of a sequence must bring a whole window (n_new = T)"); return HOLO_ERR_STATE; }
    {   // the centred projection exists only in the deflation form (rejected set at most half of the kept set)
        const int nS = c->k_hi - c->k_lo + 1;
        if (2 * (T - nS) > nS) { holo_set_error("holo_push needs a component window whose complement is at most half of it (got [%d, %d] of %d)", c->k_lo, c->k_hi, T); return HOLO_ERR_STATE; }
        if (c->push_ready == 2 && !push_ring_possible(c)) { holo_set_error("tune keys 7, 8, 10 must not change in the middle of a pipelined holo_push sequence (restart with n_new = T)"); return HOLO_ERR_STATE; }
    }
    cudaStream_t st = (cudaStream_t)stream;
    int rc;
    if (!c->Cd) HOLO_CUDA_OK(cudaMalloc(&c->Cd, (size_t)T * T * sizeof(double2)));
    const int extra = (T / 2 + 7) / 8 * 8 > 8 ? (T / 2 + 7) / 8 * 8 : 8;
    if (n_new == T) {
        // (re)start: reference = mean of this window; transform all T frames
        if ((rc = join_side(c, st, -1))) return rc;
        if ((rc = project_pending(c, st))) return rc;
        if (push_ring_possible(c)) {
            if ((rc = submit_init(c, /*second_stack=*/false))) return rc;   // side stream, events, second C / V slot (no second H)
            if (!c->ring) {
                c->ring_slots = T + extra;
                HOLO_CUDA_OK(cudaMalloc(&c->ring, (size_t)c->ring_slots * c->npix * sizeof(float2)));
                HOLO_CUDA_OK(cudaMalloc(&c->Gs, (size_t)c->ring_slots * c->ring_slots * sizeof(double)));
            }
            if ((rc = holo_launch_fresnel(c, new_frames_dev, c->ring, st))) return rc;
            c->push_ready = 2; c->ring_a = 0;
        } else {
            if ((rc = holo_launch_fresnel(c, new_frames_dev, c->H, st))) return rc;
            c->push_ready = 1; c->push_head = 0;
        }
    } else {
        if (c->push_ready == 2 && (n_new % 8 != 0 || n_new > extra)) { if ((rc = push_ring_to_flat(c, st))) return rc; }
        // overwrite the n_new oldest slots (two pieces when the range wraps around the ring)
        const int Rn = c->push_ready == 2 ? c->ring_slots : T;
        float2* base = c->push_ready == 2 ? c->ring : c->H;
        const int start = c->push_ready == 2 ? (c->ring_a + T) % Rn : c->push_head;
        if (c->push_ready == 2) { if ((rc = join_side(c, st, (int)(c->npush & 1)))) return rc; }   // readers of these slots: the push before last
        int done = 0;
        while (done < n_new) {
            const int slot = (start + done) % Rn;
            const int n = (n_new - done < Rn - slot) ? n_new - done : Rn - slot;
            if ((rc = holo_launch_fresnel(c, new_frames_dev + (size_t)done * c->npix, base + (size_t)slot * c->npix, st,
                                          /*with_sum=*/false, n))) return rc;
            done += n;
        }
        if (c->push_ready == 2) c->ring_a = (c->ring_a + n_new) % Rn;
        else c->push_head = (c->push_head + n_new) % T;
    }
    if (c->push_ready == 1) {
        // serial form: everything in stream order on ctx->H
        c->center_gram = 1;
        rc = holo_launch_covariance(c, c->H, c->C, st, /*real_only=*/true);
        c->center_gram = 0;
        if (rc) return rc;
        if ((rc = holo_launch_eig(c, c->C, c->evals, c->V, st, c->tune[HOLO_TUNE_COV_REAL] != 0))) return rc;
        return holo_launch_project(c, c->H, c->V, c->k_lo, c->k_hi, /*allow_complement=*/1, image_dev, st, /*center=*/1);
    }
    // pipelined form (same structure as holo_submit): eigensolver + projection on the side stream; the image is
    // complete after holo_flush or after the push after next
    const int s = (int)(c->npush & 1);
    // no SM split here: with only n_new transforms per window the side chain (eigensolver + projection) is the longer
    // one, and the projection is fastest on all SMs (measured at 1024^2 x 32, stride 8: 204 us vs 220 us with the split)
    const int split = 0;
    float2* C = s ? c->C1 : c->C;
    c->ring_rb0 = c->ring_a / 8; c->ring_nrb = c->ring_slots / 8;
    c->center_gram = 1;
    c->cov_grid_cap = split > 0 ? c->num_sms - split : 0;
    // incremental Gram: only the products with the new frames (kept in a slot-indexed FP64 store), when the job
    // count fits one CTA shape; a restart recomputes everything
    const int njobs_new = (T / 16) * (n_new / 8);
    c->cov_new_blocks = (n_new < T && c->tune[HOLO_TUNE_PUSH_INCR] && (njobs_new == 1 || njobs_new == 2 || njobs_new == 4 || njobs_new == 8)) ? n_new / 8 : 0;
    rc = holo_launch_covariance(c, c->ring, C, st, /*real_only=*/true);
    c->center_gram = 0; c->cov_grid_cap = 0; c->cov_new_blocks = 0;
    if (!rc) rc = cudaEventRecord(c->ev_cov[s], st) == cudaSuccess && cudaStreamWaitEvent(c->side, c->ev_cov[s], 0) == cudaSuccess ? HOLO_OK : HOLO_ERR_CUDA;
    if (!rc) {
        int32_t* status_main = c->status;
        if (s) c->status = c->status1;
        rc = holo_launch_eig(c, C, s ? c->evals1 : c->evals, s ? c->V1 : c->V, c->side, c->tune[HOLO_TUNE_COV_REAL] != 0);
        c->status = status_main;
    }
    if (!rc) {
        c->proj_grid_cap = split > 0 ? split : 0;
        rc = holo_launch_project(c, c->ring, s ? c->V1 : c->V, c->k_lo, c->k_hi, /*allow_complement=*/1, image_dev, c->side, /*center=*/1);
        c->proj_grid_cap = 0;
    }
    c->ring_rb0 = 0; c->ring_nrb = 0;
    if (rc) return rc;
    HOLO_CUDA_OK(cudaEventRecord(c->ev_proj[s], c->side));
    c->proj_recorded[s] = 1;
    c->npush++;
    return HOLO_OK;
}

// ---- streaming host entry: H2D of stack i (copy stream) runs under the kernels of stack i-1 ----------
static int host_init(holo_ctx* c) {
    if (c->copy) return HOLO_OK;
    const size_t fbytes = (size_t)c->T * c->npix * sizeof(uint16_t), ibytes = (size_t)c->npix * sizeof(float);
    for (int i = 0; i < 2; ++i) {
        HOLO_CUDA_OK(cudaMalloc(&c->fstage[i], fbytes));
        HOLO_CUDA_OK(cudaMalloc(&c->istage[i], ibytes));
        HOLO_CUDA_OK(cudaEventCreateWithFlags(&c->ev_h2d[i], cudaEventDisableTiming));
        HOLO_CUDA_OK(cudaEventCreateWithFlags(&c->ev_free[i], cudaEventDisableTiming));
    }
    HOLO_CUDA_OK(cudaStreamCreateWithFlags(&c->copy, cudaStreamNonBlocking));
    return HOLO_OK;
}

static int deliver_host(holo_ctx* c, cudaStream_t st) {      // D2H of the image whose projection was just enqueued
    if (!c->pend_image_host) return HOLO_OK;
    HOLO_CUDA_OK(cudaMemcpyAsync(c->pend_image_host, c->istage[c->pend_islot], (size_t)c->npix * sizeof(float), cudaMemcpyDeviceToHost, st));
    c->pend_image_host = nullptr;
    return HOLO_OK;
}

extern "C" int holo_submit_host(holo_ctx* c, const uint16_t* frames_host, float* image_host, holo_stream stream) {
    CHECK_CTX(c); CHECK_PTR(frames_host, "frames_host"); CHECK_PTR(image_host, "image_host");
    cudaStream_t st = (cudaStream_t)stream;
    int rc;
    if ((rc = host_init(c))) return rc;
    const size_t fbytes = (size_t)c->T * c->npix * sizeof(uint16_t);
    if (c->mode == 3) {
        // mode 3 reads the frames of stack i again in the NEXT submit (energy pass): three frame stages, so that the copy of
        // stack i+1 still runs under the kernels enqueued by this call
        if (!c->fstage[2]) {
            HOLO_CUDA_OK(cudaMalloc(&c->fstage[2], fbytes));
            HOLO_CUDA_OK(cudaEventCreateWithFlags(&c->ev_h2d[2], cudaEventDisableTiming));
            HOLO_CUDA_OK(cudaEventCreateWithFlags(&c->ev_free[2], cudaEventDisableTiming));
        }
        const long long i = c->nsubmit_host;
        const int s3 = (int)(i % 3), si = (int)(i & 1);
        if (i >= 3) HOLO_CUDA_OK(cudaStreamWaitEvent(c->copy, c->ev_free[s3], 0));           // read last by the submit of stack i-2
        HOLO_CUDA_OK(cudaMemcpyAsync(c->fstage[s3], frames_host, fbytes, cudaMemcpyHostToDevice, c->copy));
        HOLO_CUDA_OK(cudaEventRecord(c->ev_h2d[s3], c->copy));
        HOLO_CUDA_OK(cudaStreamWaitEvent(st, c->ev_h2d[s3], 0));
        if ((rc = holo_submit(c, c->fstage[s3], c->istage[si], stream))) return rc;          // enqueues the image of stack i-1
        if (i >= 1) HOLO_CUDA_OK(cudaEventRecord(c->ev_free[(int)((i - 1) % 3)], st));
        if ((rc = deliver_host(c, st))) return rc;
        c->pend_image_host = image_host; c->pend_islot = si; c->nsubmit_host++;
        HOLO_CUDA_OK(cudaEventSynchronize(c->ev_h2d[s3]));       // frames_host may be reused on return
        return HOLO_OK;
    }
    const int s = (int)(c->nsubmit_host & 1);
    if (c->nsubmit_host >= 2) HOLO_CUDA_OK(cudaStreamWaitEvent(c->copy, c->ev_free[s], 0));   // stage s was read by stack i-2
    HOLO_CUDA_OK(cudaMemcpyAsync(c->fstage[s], frames_host, fbytes, cudaMemcpyHostToDevice, c->copy));
    HOLO_CUDA_OK(cudaEventRecord(c->ev_h2d[s], c->copy));
    HOLO_CUDA_OK(cudaStreamWaitEvent(st, c->ev_h2d[s], 0));
    if (c->mode == 1 && c->tune[HOLO_TUNE_SPLIT_SMS] > 0) {
        // SM-split mode: the projection of stack i-2 (same slot) is joined first and its image copied out BEFORE
        // anything of stack i is enqueued, so the copy is ordered before the projection of stack i reuses the slot
        if ((rc = join_side(c, st, s))) return rc;
        if (c->pend_host_slot[s]) {
            HOLO_CUDA_OK(cudaMemcpyAsync(c->pend_host_slot[s], c->istage[s], (size_t)c->npix * sizeof(float), cudaMemcpyDeviceToHost, st));
            c->pend_host_slot[s] = nullptr;
        }
        if ((rc = holo_submit(c, c->fstage[s], c->istage[s], stream))) return rc;
        HOLO_CUDA_OK(cudaEventRecord(c->ev_free[s], st));
        c->pend_host_slot[s] = image_host; c->nsubmit_host++;
        HOLO_CUDA_OK(cudaEventSynchronize(c->ev_h2d[s]));
        return HOLO_OK;
    }
    if ((rc = holo_submit(c, c->fstage[s], c->istage[s], stream))) return rc;   // enqueues the projection of stack i-1
    HOLO_CUDA_OK(cudaEventRecord(c->ev_free[s], st));
    if ((rc = deliver_host(c, st))) return rc;
    c->pend_image_host = image_host; c->pend_islot = s; c->nsubmit_host++;
    HOLO_CUDA_OK(cudaEventSynchronize(c->ev_h2d[s]));        // frames_host may be reused on return
    return HOLO_OK;
}

extern "C" int holo_flush_host(holo_ctx* c, holo_stream stream) {
    CHECK_CTX(c);
    cudaStream_t st = (cudaStream_t)stream;
    int rc;
    if ((rc = holo_flush(c, stream))) return rc;
    if ((rc = deliver_host(c, st))) return rc;
    for (int k = 0; k < 2; ++k) {                       // SM-split mode: up to two images are still owed
        const int s = (int)((c->nsubmit_host + k) & 1);  // older slot first
        if (c->pend_host_slot[s]) {
            HOLO_CUDA_OK(cudaMemcpyAsync(c->pend_host_slot[s], c->istage[s], (size_t)c->npix * sizeof(float), cudaMemcpyDeviceToHost, st));
            c->pend_host_slot[s] = nullptr;
        }
    }
    HOLO_CUDA_OK(cudaStreamSynchronize(st));
    return HOLO_OK;
}

extern "C" int holo_process_host(holo_ctx* c, const uint16_t* frames_host, float* image_host, holo_stream stream) {
    CHECK_CTX(c); CHECK_PTR(frames_host, "frames_host"); CHECK_PTR(image_host, "image_host");
    cudaStream_t st = (cudaStream_t)stream;
    const size_t fbytes = (size_t)c->T * c->npix * sizeof(uint16_t), ibytes = (size_t)c->npix * sizeof(float);
    if (!c->frames_stage) {
        if (cudaMalloc(&c->frames_stage, fbytes) != cudaSuccess || cudaMalloc(&c->image_stage, ibytes) != cudaSuccess) {
            holo_set_error("staging allocation failed");
            return HOLO_ERR_ALLOC;
        }
    }
    HOLO_CUDA_OK(cudaMemcpyAsync(c->frames_stage, frames_host, fbytes, cudaMemcpyHostToDevice, st));
    int rc = holo_process(c, c->frames_stage, c->image_stage, stream);
    if (rc) return rc;
    HOLO_CUDA_OK(cudaMemcpyAsync(image_host, c->image_stage, ibytes, cudaMemcpyDeviceToHost, st));
    HOLO_CUDA_OK(cudaStreamSynchronize(st));
    return HOLO_OK;
}

extern "C" int holo_set_range(holo_ctx* c, int k_lo, int k_hi) {
    CHECK_CTX(c);
    if (k_lo < 1 || k_hi > c->T || k_lo > k_hi) { holo_set_error("need 1 <= k_lo <= k_hi <= T (got %d, %d)", k_lo, k_hi); return HOLO_ERR_ARG; }
    if (c->push_ready && 2 * (c->T - (k_hi - k_lo + 1)) > (k_hi - k_lo + 1)) {
        holo_set_error("a holo_push sequence is open: its window's complement must stay at most half of the window");
        return HOLO_ERR_STATE;
    }
    if (c->mode == 3) { const int rc3 = mode3_prepare(c, k_lo, k_hi); if (rc3) return rc3; }
    c->k_lo = k_lo; c->k_hi = k_hi;
    return HOLO_OK;
}

extern "C" int holo_set_assume_unitary(holo_ctx* c, int on) {
    CHECK_CTX_QUIET(c);
    c->assume_unitary = on ? 1 : 0;
    return HOLO_OK;
}

extern "C" const void* holo_workspace(holo_ctx* c, int which) {
    if (!c) return nullptr;
    switch (which) {
        case HOLO_WS_SUM: return c->sum;
        case HOLO_WS_H: return c->H;
        case HOLO_WS_C: return c->C;
        case HOLO_WS_EVALS: return c->evals;
        case HOLO_WS_V: return c->V;
        case HOLO_WS_STATUS: return c->status;
        case HOLO_WS_QX: return c->qx;
        case HOLO_WS_QY: return c->qy;
    }
    return nullptr;
}

extern "C" int holo_workspace_copy(holo_ctx* c, int which, void* dst_dev, unsigned long long nbytes, holo_stream stream) {
    CHECK_CTX_QUIET(c); CHECK_PTR(dst_dev, "dst_dev");
    const void* src = holo_workspace(c, which);
    if (!src) { holo_set_error("bad workspace id %d", which); return HOLO_ERR_ARG; }
    const size_t T = (size_t)c->T, np = (size_t)c->npix;
    const size_t cap[8] = {np * 4, T * np * 8, T * T * 8, T * 4, T * T * 8, 8 * 4, (size_t)c->nx * 8, (size_t)c->ny * 8};
    if (nbytes > cap[which]) { holo_set_error("workspace array %d holds %zu bytes (asked for %llu)", which, cap[which], nbytes); return HOLO_ERR_ARG; }
    HOLO_CUDA_OK(cudaMemcpyAsync(dst_dev, src, (size_t)nbytes, cudaMemcpyDeviceToDevice, (cudaStream_t)stream));
    return HOLO_OK;
}

extern "C" int holo_status(holo_ctx* c, int32_t status_host[4], holo_stream stream) {
    CHECK_CTX_QUIET(c); CHECK_PTR(status_host, "status_host");
    cudaStream_t st = (cudaStream_t)stream;
    // the eigensolvers of holo_submit / holo_push run on the side stream: join it first (the caller should have called
    // holo_flush; this only makes the read safe), then read the word of the last solve of each workspace slot
    HOLO_CUDA_OK(cudaStreamSynchronize(st));
    if (c->side) HOLO_CUDA_OK(cudaStreamSynchronize(c->side));
    HOLO_CUDA_OK(cudaMemcpyAsync(status_host, c->status, 4 * sizeof(int32_t), cudaMemcpyDeviceToHost, st));
    HOLO_CUDA_OK(cudaStreamSynchronize(st));
    if (c->status1 && !status_host[0]) {
        int32_t other[4];
        HOLO_CUDA_OK(cudaMemcpyAsync(other, c->status1, 4 * sizeof(int32_t), cudaMemcpyDeviceToHost, st));
        HOLO_CUDA_OK(cudaStreamSynchronize(st));
        if (other[0]) memcpy(status_host, other, sizeof(other));      // report the slot that failed
    }
    *(volatile int32_t*)c->noconv_host = 0;                // reported here: the next call is not refused for it
    if (status_host[0]) { holo_set_error("Jacobi eigensolver hit the sweep cap (%d sweeps)", status_host[1]); return HOLO_ERR_NOCONV; }
    return HOLO_OK;
}

extern "C" int holo_launches_per_process(holo_ctx* c) {
    CHECK_CTX_QUIET(c);
    if (c->mode == 3) {
        const int ndefl = (c->k_lo - 1) + (c->T - c->k_hi);
        const bool eigen = holo_mode3_eigen_form(c, c->k_lo, c->k_hi);
        return 2 /*sum + Gram, reduce + finish*/ + 1 /*eig*/ + ((eigen || ndefl) ? 1 : 0) + 2 /*row pass, column energy*/
             + (holo_mode3_splits(c, eigen ? c->k_hi - c->k_lo + 1 : c->T) > 1 ? 1 : 0);
    }
    if (c->mode == 2) return 2 /*sum + Gram, finish*/ + (holo_fresnel_launch_count(c) - 1) + 1 /*eig*/ + 1 /*project*/;
    return holo_fresnel_launch_count(c) + 2 /*cov partial + reduce*/ + 1 /*eig*/ + 1 /*project*/;
}

// experiment knobs (see holo_internal.cuh HOLO_TUNE_* and include/holo.h)
extern "C" int holo_tune(holo_ctx* c, int key, int value) {
    CHECK_CTX_QUIET(c);
    if (key < 0 || key >= HOLO_NUM_TUNE) { holo_set_error("bad tuning key"); return HOLO_ERR_ARG; }
    if (key == HOLO_TUNE_FFT_GROUP) {
        if (value < 1 || value > c->T) { holo_set_error("fft group out of range"); return HOLO_ERR_ARG; }
        if (value > c->scratch_frames) {
            cudaDeviceSynchronize();
            cudaFree(c->scratch);
            c->scratch = nullptr;
            if (cudaMalloc(&c->scratch, (size_t)value * c->npix * sizeof(float2)) != cudaSuccess) { holo_set_error("scratch allocation failed"); return HOLO_ERR_ALLOC; }
        }
        c->scratch_frames = value;
    }
    if (key == HOLO_TUNE_PROFILE && value && !c->prof_ev) {
        c->prof_ev = new cudaEvent_t[2 * HOLO_PROF_CAP];
        c->prof_cls = new int[HOLO_PROF_CAP];
        for (int i = 0; i < 2 * HOLO_PROF_CAP; ++i) HOLO_CUDA_OK(cudaEventCreate(&c->prof_ev[i]));
        c->prof_n = 0;
    }
    if (key == HOLO_TUNE_PDL) holo_pdl_enabled = value != 0;
    if (key == HOLO_TUNE_TILED_G && value != 0 && value != 8 && value != 16 && value != 32) { holo_set_error("tile width must be 0, 8, 16 or 32"); return HOLO_ERR_ARG; }
    if (key == HOLO_TUNE_COV_GRIDX && (value < 1 || value > c->cov_parts_cap)) { holo_set_error("cov grid out of range"); return HOLO_ERR_ARG; }
    c->tune[key] = value;
    return HOLO_OK;
}

// per-kernel-class device time accumulated since the last read, while holo_tune(ctx, 5, 1) is on.
// ms_out[HOLO_K_COUNT], count_out[HOLO_K_COUNT]; synchronises the device.
extern "C" int holo_profile_read(holo_ctx* c, double* ms_out, int* count_out) {
    CHECK_CTX_QUIET(c); CHECK_PTR(ms_out, "ms_out"); CHECK_PTR(count_out, "count_out");
    for (int k = 0; k < HOLO_K_COUNT; ++k) { ms_out[k] = 0.0; count_out[k] = 0; }
    if (!c->prof_ev) return HOLO_OK;
    HOLO_CUDA_OK(cudaDeviceSynchronize());
    for (int i = 0; i < c->prof_n; ++i) {
        float ms = 0.f;
        HOLO_CUDA_OK(cudaEventElapsedTime(&ms, c->prof_ev[2 * i], c->prof_ev[2 * i + 1]));
        ms_out[c->prof_cls[i]] += ms;
        count_out[c->prof_cls[i]] += 1;
    }
    c->prof_n = 0;
    return HOLO_OK;
}

extern "C" int holo_fft_group(holo_ctx* c) { return c ? c->scratch_frames : 0; }
