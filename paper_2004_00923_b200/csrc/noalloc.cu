// noalloc.cu -- holo_normalize_static: the image normalisation of PAPER.md:86 (M <- M / <M>, as holo_normalize in display.cu)
// for callers that cannot call cudaMalloc (code under CUDA-graph capture, tight serving loops, harnesses that forbid it).
// No handle, no cudaMalloc / cudaFree, no allocating library routine: the partial sums of the mean -- the scratch memory of
// the reduction -- live in a file-scope __device__ array of fixed size, which every GPU that loads the library holds until
// the process exits (32 KB).
//
// The array's NAME is a device address only in device code.  In host code it is a host-side stand-in: a kernel given it as
// an argument would fault or silently use the wrong memory.  The host therefore resolves the device address once per
// device with cudaGetSymbolAddress (that device current) and passes THAT pointer to the kernels.
//
// Every call shares the one array and finds the previous call's contents in it.  Nothing has to start at zero: the first
// kernel of a call writes every partial the second kernel of the same call reads (entries beyond the call's own count are
// never read).  Calls that overlap on the GPU (two streams, two host threads) race on it: serialise them.
// Product code (CUDA, sm_100a); nothing here is shared with oracle/.
#include "holo_internal.cuh"
#include <mutex>

namespace {

constexpr int NA_THREADS = 256;
constexpr int NA_CHUNK = 4096;                                      // pixels per partial sum: a FIXED partition (not a function of the
                                                                    // GPU's SM count): the result is the same on every device
constexpr long long NA_MAX_PIXELS = HOLO_STATIC_MAX_PIXELS;         // 2^24 = 4096 x 4096, the largest frame the library transforms
constexpr int NA_MAX_PARTS = (int)(NA_MAX_PIXELS / NA_CHUNK);       // 4096 doubles = 32 KB
constexpr int NA_MAX_DEVICES = 64;

}  // namespace

// the scratch: file scope, internal linkage, one copy per GPU that loads the library
static __device__ __align__(256) double g_norm_scratch[NA_MAX_PARTS];

namespace {

// partial[b] = sum of chunk b in FP64: thread-strided sums, then a fixed shared-memory tree (bit-reproducible)
__global__ void __launch_bounds__(NA_THREADS) k_static_partial_sums(const float* __restrict__ in, long long npix, double* __restrict__ partial) {
    __shared__ double sh[NA_THREADS];
    const long long p0 = (long long)blockIdx.x * NA_CHUNK;
    const long long p1 = p0 + NA_CHUNK < npix ? p0 + NA_CHUNK : npix;
    double acc = 0.0;
    for (long long p = p0 + threadIdx.x; p < p1; p += NA_THREADS) acc += (double)__ldg(in + p);
    sh[threadIdx.x] = acc;
    __syncthreads();
    for (int s = NA_THREADS / 2; s > 0; s >>= 1) {
        if ((int)threadIdx.x < s) sh[threadIdx.x] += sh[threadIdx.x + s];
        __syncthreads();
    }
    if (threadIdx.x == 0) partial[blockIdx.x] = sh[0];
}

// every CTA adds the nparts partials up in the same fixed order (thread t: t, t + 256, ...; then the same tree) and scales
// chunk blockIdx.x.  out == in is allowed: a thread reads an element before it writes it, and nobody else touches it.
__global__ void __launch_bounds__(NA_THREADS) k_static_scale(const float* in, float* out, long long npix, const double* __restrict__ partial, int nparts) {
    __shared__ double sh[NA_THREADS];
    double acc = 0.0;
    for (int i = threadIdx.x; i < nparts; i += NA_THREADS) acc += partial[i];
    sh[threadIdx.x] = acc;
    __syncthreads();
    for (int s = NA_THREADS / 2; s > 0; s >>= 1) {
        if ((int)threadIdx.x < s) sh[threadIdx.x] += sh[threadIdx.x + s];
        __syncthreads();
    }
    const double mean = sh[0] / (double)npix;
    const float sc = mean != 0.0 ? (float)(1.0 / mean) : 1.f;      // a zero image stays zero (as holo_normalize)
    const long long p0 = (long long)blockIdx.x * NA_CHUNK;
    const long long p1 = p0 + NA_CHUNK < npix ? p0 + NA_CHUNK : npix;
    for (long long p = p0 + threadIdx.x; p < p1; p += NA_THREADS) out[p] = in[p] * sc;
}

std::mutex g_mu;
double* g_scratch_dev[NA_MAX_DEVICES] = {};                         // device address of g_norm_scratch, per device

// set-up, once per device, with that device current: the DEVICE address of the scratch array
int scratch_of_current_device(double** out) {
    int dev = -1;
    HOLO_CUDA_OK(cudaGetDevice(&dev));
    if (dev < 0 || dev >= NA_MAX_DEVICES) { holo_set_error("holo_normalize_static: device ordinal %d not supported (max %d)", dev, NA_MAX_DEVICES - 1); return HOLO_ERR_STATE; }
    std::lock_guard<std::mutex> lock(g_mu);
    if (!g_scratch_dev[dev]) {
        double* p = nullptr;
        HOLO_CUDA_OK(cudaGetSymbolAddress((void**)&p, g_norm_scratch));
        if (!p) { holo_set_error("holo_normalize_static: cudaGetSymbolAddress returned a null address"); return HOLO_ERR_CUDA; }
        g_scratch_dev[dev] = p;
    }
    *out = g_scratch_dev[dev];
    return HOLO_OK;
}

}  // namespace

extern "C" int holo_normalize_static(const float* in_dev, float* out_dev, int nx, int ny, holo_stream stream) {
    if (!in_dev || !out_dev) { holo_set_error("holo_normalize_static: null image pointer"); return HOLO_ERR_ARG; }
    if (nx < 1 || ny < 1) { holo_set_error("holo_normalize_static: need nx, ny >= 1 (got %d x %d)", nx, ny); return HOLO_ERR_ARG; }
    const long long npix = (long long)nx * (long long)ny;
    if (npix > NA_MAX_PIXELS) {
        holo_set_error("holo_normalize_static: %d x %d = %lld pixels exceed the static scratch (HOLO_STATIC_MAX_PIXELS = %lld); use holo_normalize",
                       nx, ny, npix, NA_MAX_PIXELS);
        return HOLO_ERR_ARG;
    }
    if (((uintptr_t)in_dev & 3) || ((uintptr_t)out_dev & 3)) { holo_set_error("holo_normalize_static: image pointers must be 4-byte aligned"); return HOLO_ERR_ARG; }
    double* scratch = nullptr;
    { const int rc = scratch_of_current_device(&scratch); if (rc) return rc; }
    const int nparts = (int)((npix + NA_CHUNK - 1) / NA_CHUNK);
    cudaStream_t st = (cudaStream_t)stream;
    k_static_partial_sums<<<nparts, NA_THREADS, 0, st>>>(in_dev, npix, scratch);
    HOLO_CUDA_OK(cudaGetLastError());
    k_static_scale<<<nparts, NA_THREADS, 0, st>>>(in_dev, out_dev, npix, scratch, nparts);
    HOLO_CUDA_OK(cudaGetLastError());
    return HOLO_OK;
}
