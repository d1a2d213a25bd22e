// project_tc.cu -- A5 + A6 for WIDE component windows on the tensor cores (direct form; T <= 32):
//   M(p) = sum_{k in [k_lo,k_hi]} | sum_t H_t(p) V_{t,k} |^2                         (Eq. 6-7)
// With many kept components (the paper's own window keeps 20 of 32; the Fourier demodulation of Eq. 8-9
// keeps 17) the projection is a dense contraction [pixels x 2T] x [2T x 2 nS]: 2 560 real FMAs per pixel at nS = 20, which
// the FP32 kernel k_project<32,2> pays with 128 accumulator registers per thread (330 us at 1024^2 x 32).  Here:
//   * a thread owns one pixel of a 128-pixel tile: it loads H_t(p) for all t (the next tile's loads are in flight in
//     registers), splits every value into TF32 hi + lo (cvt.rna; x = hi + lo to 2^-21) and writes four K-major
//     SWIZZLE_128B operand tiles [128 pixels x T]: Re-plane and Im-plane, hi and lo;
//   * B operands, built once per CTA from V: B1 = [Re V ; Im V], B2 = [-Im V ; Re V] (rows = output columns: the nS real
//     parts, then the nS imaginary parts of P), hi and lo;
//   * D [128 pixels x 2 nS] (TMEM) = A_re B1^T + A_im B2^T with the three products hi hi + hi lo + lo hi each ("3 x TF32":
//     FP32-class accuracy; single-pass TF32 would leave 1e-4 on M);
//   * epilogue: the thread reads its pixel's row of D and stores the sum of squares -- Re and Im parts need not be told
//     apart.  P is never stored.
// Two CTAs per SM (one operand stage each, 96 KB): while one waits for its MMAs the other converts.
#include "holo_internal.cuh"
#include "tma.cuh"

namespace {

constexpr int PT_THREADS = 128;
constexpr int PT_TILE = 128 * 128;                 // bytes: 128 rows x 128 B (32 floats of K)
constexpr int PT_SMEM = 1024 + 4 * PT_TILE + 4 * (64 * 128) + 64;

__device__ __forceinline__ uint64_t pt_sdesc(uint32_t saddr) {
    // K-major, SWIZZLE_128B canonical layout: 8-row atoms of 1024 B (SBO = 1024), LBO = 16 B, descriptor version 1 (sm_100)
    return (uint64_t)((saddr & 0x3FFFFu) >> 4) | ((uint64_t)1 << 16) | ((uint64_t)(1024 >> 4) << 32) | ((uint64_t)1 << 46) | ((uint64_t)2 << 61);
}
__device__ __forceinline__ void pt_mma(uint32_t tmem_d, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t accumulate) {
    asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
                 "tcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n\t}"
                 ::"r"(tmem_d), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate) : "memory");
}
__device__ __forceinline__ float pt_tf32(float x) {
    uint32_t r;
    asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(r) : "f"(x));
    return __uint_as_float(r);
}
__device__ __forceinline__ uint32_t pt_off(int row, int j16) {    // byte offset of 16-byte chunk j16 of row `row` in a tile
    return (uint32_t)(row >> 3) * 1024u + (uint32_t)(row & 7) * 128u + (uint32_t)((j16 ^ (row & 7)) << 4);
}

// H complex64 [T][npix]; V complex64 [T][T] row-major (column = component); columns c_lo .. c_lo + nS - 1 are kept
__global__ void __launch_bounds__(PT_THREADS, 2)
k_project_tc(const float2* __restrict__ H, const float2* __restrict__ V, float* __restrict__ M, long long npix, int T, int c_lo, int nS) {
    extern __shared__ unsigned char smraw_[];
    const uint32_t s0 = smem_u32(smraw_);
    const uint32_t pad = (1024u - (s0 & 1023u)) & 1023u;
    unsigned char* base = smraw_ + pad;
    const uint32_t sbase = s0 + pad;
    // A tiles: [0] Re hi, [1] Re lo, [2] Im hi, [3] Im lo; then B tiles (64 rows x 128 B each): B1 hi, B1 lo, B2 hi, B2 lo
    unsigned char* Bt = base + 4 * PT_TILE;
    uint64_t* mma_done = reinterpret_cast<uint64_t*>(Bt + 4 * 64 * 128);
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(mma_done + 1);
    const int tid = threadIdx.x, warp = tid >> 5;
    const int N = ((2 * nS + 15) / 16) * 16;                  // MMA N: multiple of 16, <= 64

    for (int i = tid; i < (4 * PT_TILE + 4 * 64 * 128) / 16; i += PT_THREADS) reinterpret_cast<uint4*>(base)[i] = make_uint4(0, 0, 0, 0);
    if (tid == 0) {
        mbar_init(mma_done, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(tmem_slot)), "r"(64) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    __syncthreads();
    // B operands (rows n = output columns; K = t): n < nS: Re P of component c_lo + n, nS <= n < 2 nS: Im P
    for (int e = tid; e < 2 * nS * 32; e += PT_THREADS) {
        const int n = e >> 5, t = e & 31;
        float b1 = 0.f, b2 = 0.f;
        if (t < T) {
            const float2 v = V[t * T + c_lo + (n < nS ? n : n - nS)];
            b1 = n < nS ? v.x : v.y;                           // multiplies Re H
            b2 = n < nS ? -v.y : v.x;                          // multiplies Im H
        }
        const uint32_t off = pt_off(n, t >> 2) + (uint32_t)(t & 3) * 4u;
        const float h1 = pt_tf32(b1), h2 = pt_tf32(b2);
        *reinterpret_cast<float*>(Bt + 0 * 8192 + off) = h1;
        *reinterpret_cast<float*>(Bt + 1 * 8192 + off) = pt_tf32(b1 - h1);
        *reinterpret_cast<float*>(Bt + 2 * 8192 + off) = h2;
        *reinterpret_cast<float*>(Bt + 3 * 8192 + off) = pt_tf32(b2 - h2);
    }
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const uint32_t tmem = *tmem_slot;
    // D = F32, A = B = TF32, K-major, M = 128
    const uint32_t idesc = (1u << 4) | (2u << 7) | (2u << 10) | ((uint32_t)(N >> 3) << 17) | ((uint32_t)(128 >> 4) << 24);

    const long long ntiles = npix / 128;
    float2 w[32], wn[32];
    auto load_tile = [&](long long tile, float2* dst) {
        const float2* src = H + tile * 128 + tid;
#pragma unroll
        for (int t = 0; t < 32; ++t) dst[t] = t < T ? __ldg(src + (size_t)t * (size_t)npix) : make_float2(0.f, 0.f);
    };
    uint32_t ph = 0u;
    if ((long long)blockIdx.x < ntiles) load_tile(blockIdx.x, wn);
    for (long long tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
#pragma unroll
        for (int t = 0; t < 32; ++t) w[t] = wn[t];
        if (tile + gridDim.x < ntiles) load_tile(tile + gridDim.x, wn);
        // the thread's pixel = row `tid` of the four A tiles; chunk j holds t = 4 j .. 4 j + 3
#pragma unroll
        for (int j = 0; j < 8; ++j) {
            const uint32_t off = pt_off(tid, j);
            float4 rh, rl, ih, il;
            rh.x = pt_tf32(w[4 * j].x); rh.y = pt_tf32(w[4 * j + 1].x); rh.z = pt_tf32(w[4 * j + 2].x); rh.w = pt_tf32(w[4 * j + 3].x);
            ih.x = pt_tf32(w[4 * j].y); ih.y = pt_tf32(w[4 * j + 1].y); ih.z = pt_tf32(w[4 * j + 2].y); ih.w = pt_tf32(w[4 * j + 3].y);
            rl.x = pt_tf32(w[4 * j].x - rh.x); rl.y = pt_tf32(w[4 * j + 1].x - rh.y); rl.z = pt_tf32(w[4 * j + 2].x - rh.z); rl.w = pt_tf32(w[4 * j + 3].x - rh.w);
            il.x = pt_tf32(w[4 * j].y - ih.x); il.y = pt_tf32(w[4 * j + 1].y - ih.y); il.z = pt_tf32(w[4 * j + 2].y - ih.z); il.w = pt_tf32(w[4 * j + 3].y - ih.w);
            *reinterpret_cast<float4*>(base + 0 * PT_TILE + off) = rh;
            *reinterpret_cast<float4*>(base + 1 * PT_TILE + off) = rl;
            *reinterpret_cast<float4*>(base + 2 * PT_TILE + off) = ih;
            *reinterpret_cast<float4*>(base + 3 * PT_TILE + off) = il;
        }
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");     // the tensor core reads the tiles through the async proxy
        asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
        __syncthreads();
        if (tid == 0) {
            asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
            const uint32_t bb = sbase + 4 * PT_TILE;
            uint32_t accum = 0u;
#pragma unroll
            for (int plane = 0; plane < 2; ++plane)            // Re H with B1, Im H with B2
#pragma unroll
                for (int k = 0; k < 4; ++k) {                  // K = 8 frames per instruction: 32 bytes further into the 128-byte rows
                    const uint64_t ah = pt_sdesc(sbase + (uint32_t)(2 * plane) * PT_TILE + (uint32_t)k * 32u);
                    const uint64_t al = pt_sdesc(sbase + (uint32_t)(2 * plane + 1) * PT_TILE + (uint32_t)k * 32u);
                    const uint64_t bh = pt_sdesc(bb + (uint32_t)(2 * plane) * 8192u + (uint32_t)k * 32u);
                    const uint64_t bl = pt_sdesc(bb + (uint32_t)(2 * plane + 1) * 8192u + (uint32_t)k * 32u);
                    pt_mma(tmem, ah, bh, idesc, accum); accum = 1u;
                    pt_mma(tmem, ah, bl, idesc, 1u);
                    pt_mma(tmem, al, bh, idesc, 1u);
                }
            asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(mma_done)) : "memory");
        }
        mbar_wait(mma_done, ph); ph ^= 1u;
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        float sum = 0.f;
        for (int c0 = 0; c0 < N; c0 += 16) {
            uint32_t r[16];
            asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
                         : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]),
                           "=r"(r[8]), "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
                         : "r"(tmem + ((uint32_t)(32 * warp) << 16) + (uint32_t)c0));
            asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
            for (int i = 0; i < 16; ++i) { const float x = __uint_as_float(r[i]); sum = fmaf(x, x, sum); }
        }
        M[tile * 128 + tid] = sum;
        asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
        __syncthreads();                                       // the accumulators and the A tiles are free again
    }
    __syncthreads();
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "r"(64) : "memory");
}

}  // namespace

bool holo_project_tc_supported(const holo_ctx* c, int nS) { return c->T <= 32 && nS >= 1 && nS <= 32 && c->npix % 128 == 0; }

int holo_launch_project_tc(holo_ctx* c, const float2* H, const float2* V, int k_lo, int k_hi, float* image, cudaStream_t st) {
    int rc;
    if ((rc = holo_ensure_smem_attr((const void*)k_project_tc, c->device, PT_SMEM))) return rc;
    const long long ntiles = c->npix / 128;
    const int cap = c->proj_grid_cap > 0 ? 2 * c->proj_grid_cap : 2 * c->num_sms;
    const int grid = (int)(ntiles < cap ? ntiles : cap);
    HoloProf prof(c, HOLO_K_PROJECT, st);
    k_project_tc<<<grid, PT_THREADS, PT_SMEM, st>>>(H, V, image, c->npix, c->T, k_lo - 1, k_hi - k_lo + 1);
    HOLO_CUDA_OK(cudaGetLastError());
    return HOLO_OK;
}
