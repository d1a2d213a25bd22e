// rawgram.cu -- mode 2 (SURVEY.md 8(f)-2 stage 1, reading c-12): the covariance of Eq. 4 from the RAW
// frames.  H_t = F[q d_t] with q unimodular and F unitary up to nx ny, so
//     C_ts = sum_p conj(H_t(p)) H_s(p) = nx ny sum_x d_t(x) d_s(x),      d_t = I_t - mean_t I,
// an exact identity.  With the integer frame sum S = sum_t I_t:  T^2 sum_x d_t d_s = T^2 G_ts - T (r_t + r_s) + tau,
// G_ts = sum_x I_t I_s (the Gram of the raw uint16 frames), r_t = sum_s G_ts, tau = sum_t r_t -- all integers.
//
// G is a dense contraction over 10^6 pixels and runs on the 5th-generation tensor cores, EXACTLY: every uint16 pixel is
// split into its two bytes, X = [hi_0 .. hi_{T-1}; lo_0 .. lo_{T-1}] (2T rows of u8, K = pixels), and
// X X^T (tcgen05.mma kind::i8, u8 x u8 -> s32 accumulators in TMEM) holds the four blocks HH, HL, LH, LL with
// G = 65536 HH + 256 (HL + LH) + LL.  One pass over the frames (2 T N_p bytes, the same read the temporal sum A0 needs):
// the kernel also writes S.  No rounding anywhere before the final conversion of C to float.
//   k_sum_gram   : persistent CTAs of 128 threads; a thread owns 2 adjacent pixels, loads them of all T frames (the loads of
//                  the next block are issued before the current one is processed), adds
//                  them up (S) and writes their bytes into the K-major SWIZZLE_128B operand tile ([128 rows x 128 B] per 128
//                  pixels, two tiles per stage, two stages); one thread issues the MMAs (M = 128, N = 64 or 128,
//                  K = 32 per instruction) and commits them to the stage's mbarrier; the s32 accumulators are drained
//                  (tcgen05.ld) into the global int64 byte-plane Gram with integer atomics before they can overflow
//                  (every 16384 pixels) and at the end.
//   k_gram_reduce_finish: one warp per entry adds the per-CTA slots up; the last CTA assembles G (int64), centres it in
//                  __int128 and writes C (float2, Im = 0).
#include "holo_internal.cuh"
#include "tma.cuh"

namespace {

constexpr int RG_THREADS = 128;
constexpr int RG_PIX = 2 * RG_THREADS;             // pixels per stage (two K tiles of 128 pixels)
constexpr int RG_TILE = 128 * 128;                 // bytes of one operand tile: 128 rows x 128 B
constexpr int RG_STAGE = 2 * RG_TILE;
constexpr int RG_SMEM = 1024 + 2 * RG_STAGE + 64 + 2 * 64 * 16;
constexpr int RG_FLUSH_ITERS = 64;                 // 64 x 256 pixels x 255^2 < 2^31

__device__ __forceinline__ uint64_t make_sdesc(uint32_t saddr) {
    // K-major, SWIZZLE_128B canonical layout: 8-row atoms of 1024 B (SBO = 1024), LBO = 16 B, descriptor version 1 (sm_100)
    return (uint64_t)((saddr & 0x3FFFFu) >> 4) | ((uint64_t)1 << 16) | ((uint64_t)(1024 >> 4) << 32) | ((uint64_t)1 << 46) | ((uint64_t)2 << 61);
}
__device__ __forceinline__ void umma_i8(uint32_t tmem_d, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t accumulate) {
    asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
                 "tcgen05.mma.cta_group::1.kind::i8 [%0], %1, %2, %3, p;\n\t}"
                 ::"r"(tmem_d), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate) : "memory");
}
__device__ __forceinline__ void umma_commit(uint64_t* bar) {
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
}
// 32 lanes x 32 bit, 16 consecutive columns: thread t of warp w gets row 32 w + t
__device__ __forceinline__ void tmem_ld16(uint32_t taddr, int32_t* v) {
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
                 : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]),
                   "=r"(v[8]), "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15])
                 : "r"(taddr));
    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
}

// frames uint16 [T][npix]; sum uint32 [npix]; X int64 [lower-triangle entries of the 2 TP x 2 TP byte-plane Gram][CTAs]: every
// CTA writes its own slot (integer sums: exact and order independent, hence deterministic).
// Thread mapping of a 256-pixel stage: thread = (pixel quad q = tid % 64, frame parity h = tid / 64); it loads its four
// pixels (8 bytes) of the frames t = 2 i + h, splits them into the two byte planes with two PRMTs and stores one 32-bit
// word per plane row; the operand-tile addresses are four per-thread bases + immediates.  The two threads of a quad
// combine their partial frame sums through shared memory (double-buffered by stage, ordered by the stage's barrier).
// FULL: T == TP (no predicates on the loads).
template <int TP, bool FULL>
__global__ void __launch_bounds__(RG_THREADS, 3)
k_sum_gram(const uint16_t* __restrict__ frames, uint32_t* __restrict__ sum, unsigned long long* __restrict__ X,
           long long npix, int T, unsigned int* __restrict__ counters) {
    constexpr int Tp = TP, NI = TP / 2;                       // NI frames per thread
    constexpr bool PF = TP <= 32;                             // next block prefetched in registers (would spill at TP = 64)
    extern __shared__ unsigned char smraw_[];
    const uint32_t s0 = smem_u32(smraw_);
    const uint32_t pad = (1024u - (s0 & 1023u)) & 1023u;
    unsigned char* base = smraw_ + pad;                       // 1024-byte aligned operand stages
    const uint32_t sbase = s0 + pad;
    uint64_t* mma_done = reinterpret_cast<uint64_t*>(base + 2 * RG_STAGE);
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(mma_done + 2);
    uint4* sscr = reinterpret_cast<uint4*>(base + 2 * RG_STAGE + 64);          // [2][64] partial frame sums of the h = 1 threads
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int N = 2 * Tp;                                     // MMA N (64 or 128); M = 128 always

    if (blockIdx.x == 0 && tid < 2 * T + 1) counters[tid] = 0u;   // ticket / completion counters of the Fresnel kernel (as k_frame_sum)
    if (blockIdx.x == 0 && tid == 0) counters[1001] = 0u;
    // rows that no frame writes (t >= T within a plane, and rows >= 2 Tp) must read as zero: clear both stages once
    for (int i = tid; i < 2 * RG_STAGE / 16; i += RG_THREADS) reinterpret_cast<uint4*>(base)[i] = make_uint4(0, 0, 0, 0);
    if (tid == 0) {
        mbar_init(mma_done + 0, 1); mbar_init(mma_done + 1, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(tmem_slot)), "r"(N) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const uint32_t tmem = *tmem_slot;
    const uint32_t idesc = (2u << 4) | ((uint32_t)(N >> 3) << 17) | ((uint32_t)(128 >> 4) << 24);   // s32 += u8 x u8, K-major A and B

    // operand tile addressing: pixel k of a tile, row r: byte (r / 8) * 1024 + (r % 8) * 128 + (((k / 16) ^ (r % 8)) * 16) + k % 16
    const int q = tid & 63, h = tid >> 6;
    const int kin = (4 * q) & 127;                            // first of the thread's four pixels inside its tile
    uint32_t rowoff[4];                                       // row t = 2 i + h: variant v = i % 4, + (i / 4) * 1024 (+ plane offset)
#pragma unroll
    for (int v = 0; v < 4; ++v) {
        const int r7 = 2 * v + h;
        rowoff[v] = (uint32_t)((q >> 5) * RG_TILE + r7 * 128 + ((((kin >> 4) ^ r7) << 4) | (kin & 15)));
    }
    const long long nblocks = (npix + RG_PIX - 1) / RG_PIX;   // npix is a multiple of 256 for every supported frame size
    uint32_t ph[2] = {0u, 0u};
    int pending[2] = {0, 0}, since_flush = 0;

    // accumulators -> this CTA's own slot of the partial store Xp[lower-triangle entry][CTA] (plain stores: the per-entry
    // 64-bit atomics of 444 CTAs on 2080 addresses cost 40 % of the kernel); k_gram_reduce_finish adds the slots up
    bool first_drain = true;
    auto drain = [&]() {                                      // (all MMAs have completed)
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        const int row = 32 * warp + lane;                     // TMEM lane = row of D
        for (int c0 = 0; c0 < N; c0 += 16) {
            int32_t v[16];
            tmem_ld16(tmem + ((uint32_t)(32 * warp) << 16) + (uint32_t)c0, v);
            if (row < N) {
                long long* dst = reinterpret_cast<long long*>(X) + ((size_t)row * (row + 1) / 2 + c0) * gridDim.x + blockIdx.x;
#pragma unroll
                for (int j = 0; j < 16; ++j)
                    if (c0 + j <= row) {
                        long long* qd = dst + (size_t)j * gridDim.x;
                        *qd = first_drain ? (long long)v[j] : *qd + (long long)v[j];
                    }
            }
        }
        first_drain = false;
        asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    };

    const size_t fstep = (size_t)2 * (size_t)npix;            // elements between two frames of a thread
    auto load_block = [&](long long blk, uint2* dst) {
        const uint16_t* src = frames + (size_t)h * (size_t)npix + (size_t)blk * RG_PIX + 4 * q;
#pragma unroll
        for (int i = 0; i < NI; ++i) {
            if (FULL || 2 * i + h < T) dst[i] = __ldg(reinterpret_cast<const uint2*>(src));
            else dst[i] = make_uint2(0u, 0u);
            src += fstep;
        }
    };
    // one stage: byte planes of block `blk` (registers w) -> operand stage s, frame sums, MMAs
    auto process = [&](const uint2* w, long long blk, int s) {
        if (pending[s]) { mbar_wait(mma_done + s, ph[s]); ph[s] ^= 1u; pending[s] = 0; }   // the MMAs that read this stage
        unsigned char* st = base + (size_t)s * RG_STAGE;
        uint32_t a0 = 0u, a1 = 0u, a2 = 0u, a3 = 0u;
#pragma unroll
        for (int i = 0; i < NI; ++i) {
            const uint2 x = w[i];
            a0 += x.x & 0xffffu; a1 += x.x >> 16; a2 += x.y & 0xffffu; a3 += x.y >> 16;
            const uint32_t lo = __byte_perm(x.x, x.y, 0x6420), hi = __byte_perm(x.x, x.y, 0x7531);
            unsigned char* p = st + rowoff[i & 3] + (i >> 2) * 1024;               // row 2 i + h of the hi plane
            *reinterpret_cast<uint32_t*>(p) = hi;
            *reinterpret_cast<uint32_t*>(p + (Tp >> 3) * 1024) = lo;             // row Tp + 2 i + h
        }
        if (h) sscr[s * 64 + q] = make_uint4(a0, a1, a2, a3);
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");     // the tensor core reads the tile through the async proxy
        asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
        __syncthreads();
        if (!h) {
            const uint4 o = sscr[s * 64 + q];
            *reinterpret_cast<uint4*>(sum + blk * RG_PIX + 4 * q) = make_uint4(a0 + o.x, a1 + o.y, a2 + o.z, a3 + o.w);
        }
        if (tid == 0) {
            asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
            const uint32_t sa0 = sbase + (uint32_t)s * RG_STAGE;
#pragma unroll
            for (int kt = 0; kt < 2; ++kt)
#pragma unroll
                for (int k = 0; k < 4; ++k) {                  // K = 32 pixels per instruction: 32 bytes further into the 128-byte rows
                    const uint64_t d = make_sdesc(sa0 + (uint32_t)kt * RG_TILE + (uint32_t)k * 32u);
                    umma_i8(tmem, d, d, idesc, (since_flush | kt | k) ? 1u : 0u);
                }
            umma_commit(mma_done + s);
        }
        pending[s] = 1;
        if (++since_flush == RG_FLUSH_ITERS) {                 // before the s32 accumulators can overflow
            for (int k = 0; k < 2; ++k) if (pending[k]) { mbar_wait(mma_done + k, ph[k]); ph[k] ^= 1u; pending[k] = 0; }
            drain();
            __syncthreads();
            since_flush = 0;
        }
    };

    // software pipeline, unrolled by two: block n + 1 is in flight (NI loads per thread) while block n is processed
    uint2 wa[NI], wb[NI];
    const long long g = gridDim.x;
    long long blk = blockIdx.x;
    if (blk < nblocks) load_block(blk, wa);
    while (blk < nblocks) {
        if (PF && blk + g < nblocks) load_block(blk + g, wb);
        process(wa, blk, 0);
        blk += g;
        if (blk >= nblocks) break;
        if (!PF) load_block(blk, wb);
        if (PF && blk + g < nblocks) load_block(blk + g, wa);
        process(wb, blk, 1);
        blk += g;
        if (!PF && blk < nblocks) load_block(blk, wa);
    }
    for (int k = 0; k < 2; ++k) if (pending[k]) { mbar_wait(mma_done + k, ph[k]); ph[k] ^= 1u; pending[k] = 0; }
    if (since_flush || first_drain) drain();
    __syncthreads();
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "r"(N) : "memory");
}

// Xp[entry][part] -> X[row][col] (lower triangle of the byte-plane Gram, int64): one warp per entry (integer sums: exact,
// order independent).  The CTA that finishes last then assembles G = 65536 HH + 256 (HL + LH) + LL (int64), centres it in
// __int128,  C = (nx ny / T^2) (T^2 G - T (r_t + r_s) + tau),  and writes the full symmetric matrix (Im = 0), rounded once.
// G < 2^57 and r < 2^63 fit int64 for every supported size.
__global__ void __launch_bounds__(256) k_gram_reduce_finish(const long long* __restrict__ Xp, int nparts, int N, unsigned long long* __restrict__ X,
                                                            unsigned int* __restrict__ done, int T, int Tp, double scale, float2* __restrict__ C) {
    __shared__ long long G[HOLO_MAX_T * HOLO_MAX_T];
    __shared__ long long r[HOLO_MAX_T];
    __shared__ long long tau_lo; __shared__ long long tau_hi;   // tau as a 128-bit value
    __shared__ int s_last;
    pdl_trigger();                                        // (the single-CTA eigensolver that follows waits for this whole kernel)
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int entry = blockIdx.x * 8 + warp;
    const int nent = N * (N + 1) / 2;
    if (entry < nent) {
        const long long* src = Xp + (size_t)entry * nparts;
        long long acc = 0;
        for (int i = lane; i < nparts; i += 32) acc += src[i];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
        if (lane == 0) {
            int row = (int)((sqrtf(8.f * (float)entry + 1.f) - 1.f) * 0.5f);
            while ((row + 1) * (row + 2) / 2 <= entry) ++row;
            while (row * (row + 1) / 2 > entry) --row;
            X[(size_t)row * N + (entry - row * (row + 1) / 2)] = (unsigned long long)acc;
        }
    }
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) s_last = atomicAdd(done, 1u) == gridDim.x - 1;
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    if (threadIdx.x == 0) *done = 0u;                          // ready for the next launch
    auto Xs = [&](int i, int j) -> long long { return (long long)__ldcg(i >= j ? X + (size_t)i * N + j : X + (size_t)j * N + i); };
    for (int e0 = 0; e0 < T * T; e0 += 4 * 256) {
        long long v[4][4];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const int e = e0 + u * 256 + threadIdx.x;
            if (e < T * T) {
                const int t = e / T, s = e - t * T;
                v[u][0] = Xs(t, s); v[u][1] = Xs(t, Tp + s); v[u][2] = Xs(Tp + t, s); v[u][3] = Xs(Tp + t, Tp + s);
            }
        }
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const int e = e0 + u * 256 + threadIdx.x;
            if (e < T * T) G[e] = v[u][0] * 65536 + (v[u][1] + v[u][2]) * 256 + v[u][3];
        }
    }
    __syncthreads();
    for (int t = warp; t < T; t += 8) {                        // row sums: one warp per row
        long long acc = 0;
        for (int s = lane; s < T; s += 32) acc += G[t * T + s];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
        if (lane == 0) r[t] = acc;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        __int128 tau = 0;
        for (int t = 0; t < T; ++t) tau += r[t];
        tau_lo = (long long)(unsigned long long)tau; tau_hi = (long long)(tau >> 64);
    }
    __syncthreads();
    const __int128 tau = ((__int128)tau_hi << 64) | (unsigned __int128)(unsigned long long)tau_lo;
    for (int e = threadIdx.x; e < T * T; e += blockDim.x) {
        const int t = e / T, s = e - t * T;
        const __int128 v = (__int128)(T * T) * G[e] - (__int128)T * ((__int128)r[t] + r[s]) + tau;     // = T^2 sum_x d_t d_s, exact
        const bool neg = v < 0;
        const unsigned __int128 a = neg ? (unsigned __int128)(-v) : (unsigned __int128)v;
        double dv = (double)(unsigned long long)(a >> 64) * 18446744073709551616.0 + (double)(unsigned long long)a;
        if (neg) dv = -dv;
        C[e] = make_float2((float)(dv * scale), 0.f);
    }
}

}  // namespace

// S = sum_t I_t (ctx->sum) and C = H^H H of the holograms these frames WOULD give, without forming them.
// finish = false: only the pass over the frames (S and the per-CTA partials of the byte-plane Gram); the caller then runs
// holo_launch_gram_finish, possibly on another stream ordered after `st` (the streaming forms put it in front of the
// eigensolver on the side stream, off the main stream's critical path)
int holo_launch_sum_gram(holo_ctx* c, const uint16_t* frames, float2* C, cudaStream_t st, bool finish) {
    const int T = c->T, Tp = T <= 32 ? 32 : 64;
    if (c->npix % RG_PIX != 0) { holo_set_error("raw-frame Gram needs nx*ny to be a multiple of %d", RG_PIX); return HOLO_ERR_ARG; }
    const long long nblocks = c->npix / RG_PIX;
    int grid = 3 * c->num_sms;                               // three CTAs per SM (64 KB of operand stages each)
    if ((long long)grid > nblocks) grid = (int)nblocks;
    int rc;
    {
        HoloProf prof(c, HOLO_K_SUM, st);
        auto launch = [&](auto kern) -> int {
            if ((rc = holo_ensure_smem_attr((const void*)kern, c->device, RG_SMEM))) return rc;
            kern<<<grid, RG_THREADS, RG_SMEM, st>>>(frames, c->sum, c->gram_Xp, c->npix, T, c->counters);
            return HOLO_OK;
        };
        if (Tp == 32) rc = T == 32 ? launch(k_sum_gram<32, true>) : launch(k_sum_gram<32, false>);
        else          rc = T == 64 ? launch(k_sum_gram<64, true>) : launch(k_sum_gram<64, false>);
        if (rc) return rc;
    }
    HOLO_CUDA_OK(cudaGetLastError());
    c->gram_nparts = grid;
    return finish ? holo_launch_gram_finish(c, C, st) : HOLO_OK;
}

int holo_launch_gram_finish(holo_ctx* c, float2* C, cudaStream_t st) {
    const int T = c->T, Tp = T <= 32 ? 32 : 64, N = 2 * Tp;
    HoloProf prof(c, HOLO_K_COV_REDUCE, st);
    const int nent = N * (N + 1) / 2;
    k_gram_reduce_finish<<<(nent + 7) / 8, 256, 0, st>>>(reinterpret_cast<const long long*>(c->gram_Xp), c->gram_nparts, N, c->gram_X, c->counters + 1000,
                                                         T, Tp, (double)c->npix / ((double)T * (double)T), C);
    HOLO_CUDA_OK(cudaGetLastError());
    return HOLO_OK;
}
