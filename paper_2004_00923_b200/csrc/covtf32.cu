// covtf32.cu -- SURVEY.md 8(f)-4: the covariance of Eq. 4 on the 5th-generation tensor cores in TF32,
// for the case north_star names ("tensor cores only if the contraction measurably pays at T >= 64 while meeting
// tolerance").  Real form only (R21: the covariance of holograms of real frames is real), i.e. the Gram of the
// stack viewed as T rows of 2 N_p floats:  C_ts = sum_k X_t[k] X_s[k].
//   * operands: the threads load the stack from global memory (16-byte loads, the next stage prefetched in registers),
//     round every value to TF32 with cvt.rna (the tensor core itself would TRUNCATE the low 13 bits: a 5e-4 bias on every
//     product, i.e. on every eigenvalue) and store it into the K-major SWIZZLE_128B operand tile.  SPLIT = true keeps the
//     rounding residual in a second tile (x = hi + lo) and issues hi hi^T + hi lo^T + lo hi^T ("3 x TF32").
//   * the tile has 128 rows but T <= 64 frames: the rows are filled with 128 / TP consecutive K-slices of the stack
//     ([X(slice 0); X(slice 1); ...]), A = B = the same tile, M = N = 128: the diagonal TP x TP blocks of D are the Grams of
//     the slices (the off-diagonal blocks are cross products of different pixels and are ignored).  No zero rows are moved.
//   * accumulators: two 128-column buffers in TMEM; every `drain_every` stages the MMAs switch buffers and the threads add
//     the finished one to FP64 registers (FP32 accumulation in the tensor core is only trusted over a few hundred products).
//   * one FP64 partial per CTA -> cov_partials (float2, Im = 0) -> the fixed-order reduction of covariance.cu.
#include "holo_internal.cuh"
#include "tma.cuh"

namespace {

constexpr int CT_THREADS = 256;
constexpr int CT_TILE = 128 * 128;                 // bytes of one operand tile: 128 rows x 128 B (32 floats of K)

__device__ __forceinline__ uint64_t ct_sdesc(uint32_t saddr) {
    // K-major, SWIZZLE_128B canonical layout: 8-row atoms of 1024 B (SBO = 1024), LBO = 16 B, descriptor version 1 (sm_100)
    return (uint64_t)((saddr & 0x3FFFFu) >> 4) | ((uint64_t)1 << 16) | ((uint64_t)(1024 >> 4) << 32) | ((uint64_t)1 << 46) | ((uint64_t)2 << 61);
}
__device__ __forceinline__ void umma_tf32(uint32_t tmem_d, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t accumulate) {
    asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
                 "tcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n\t}"
                 ::"r"(tmem_d), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate) : "memory");
}
__device__ __forceinline__ void ct_commit(uint64_t* bar) {
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void tmem_ld16f(uint32_t taddr, float* v) {
    uint32_t r[16];
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]),
                   "=r"(r[8]), "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
                 : "r"(taddr));
    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
    for (int i = 0; i < 16; ++i) v[i] = __uint_as_float(r[i]);
}
__device__ __forceinline__ float to_tf32(float x) {
    uint32_t r;
    asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(r) : "f"(x));
    return __uint_as_float(r);
}

template <int TP, bool SPLIT>
__global__ void __launch_bounds__(CT_THREADS, 1)
k_cov_tf32(const float2* __restrict__ H, float2* __restrict__ partials, long long npix, int T, int T8, int drain_every) {
    constexpr int S = 128 / TP;                       // K-slices stacked in the 128 rows of a tile
    constexpr int TILES = SPLIT ? 2 : 4;              // K-tiles per stage
    constexpr int FPF = TILES * S * 32;               // floats of one frame per stage
    constexpr int PIX = FPF / 2;                      // pixels per stage
    constexpr int CPF = FPF / 4;                      // 16-byte chunks of one frame per stage
    constexpr int STAGE = TILES * CT_TILE * (SPLIT ? 2 : 1);
    constexpr int TSTEP = CT_THREADS / CPF;           // frames between two items of a thread
    constexpr int ITEMS = TP / TSTEP;                 // items (frame, chunk) per thread per stage
    extern __shared__ unsigned char smraw_[];
    const uint32_t s0 = smem_u32(smraw_);
    const uint32_t pad = (1024u - (s0 & 1023u)) & 1023u;
    unsigned char* base = smraw_ + pad;               // 1024-byte aligned operand stages
    const uint32_t sbase = s0 + pad;
    uint64_t* mma_done = reinterpret_cast<uint64_t*>(base + 2 * STAGE);
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(mma_done + 2);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;

    for (int i = tid; i < 2 * STAGE / 16; i += CT_THREADS) reinterpret_cast<uint4*>(base)[i] = make_uint4(0, 0, 0, 0);   // rows t >= T stay zero
    if (tid == 0) {
        mbar_init(mma_done + 0, 1); mbar_init(mma_done + 1, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(tmem_slot)), "r"(256) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const uint32_t tmem = *tmem_slot;
    // D = F32, A = B = TF32, K-major, N = 128, M = 128
    const uint32_t idesc = (1u << 4) | (2u << 7) | (2u << 10) | ((uint32_t)(128 >> 3) << 17) | ((uint32_t)(128 >> 4) << 24);

    // the thread's items of a stage: chunk c of frames t0, t0 + TSTEP, ...
    const int c = tid % CPF, t0 = tid / CPF;
    const int f = 4 * c;                               // first float of the chunk inside the frame's FPF floats of the stage
    const int ktile = f / (S * 32), slice = (f % (S * 32)) / 32, j16 = c & 7;
    const long long nblocks = npix / PIX;              // npix is a multiple of 256 >= PIX for every supported frame size
    uint32_t ph[2] = {0u, 0u};
    int it = 0, pending[2] = {0, 0};

    // FP64 accumulators of the thread's part of D: row r = 32 (warp % 4) + lane (slice r / TP, frame r % TP), columns
    // r / TP * TP + (warp / 4) * TP / 2 + [0, TP / 2)
    constexpr int NACC = TP / 2;
    double acc[NACC];
#pragma unroll
    for (int i = 0; i < NACC; ++i) acc[i] = 0.0;
    const int drow = 32 * (warp & 3) + lane;
    const int dcol0 = (drow / TP) * TP + (warp >> 2) * NACC;
    auto drain = [&](int buf) {
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
#pragma unroll
        for (int q = 0; q < NACC / 16; ++q) {
            float v[16];
            tmem_ld16f(tmem + ((uint32_t)(32 * (warp & 3)) << 16) + (uint32_t)(buf * 128 + dcol0 + 16 * q), v);
#pragma unroll
            for (int i = 0; i < 16; ++i) acc[16 * q + i] += (double)v[i];
        }
        asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    };

    float4 w[ITEMS], wn[ITEMS];
    auto load_block = [&](long long blk, float4* dst) {
        const float4* src = reinterpret_cast<const float4*>(H + blk * PIX) + c;
#pragma unroll
        for (int i = 0; i < ITEMS; ++i) {
            const int t = t0 + i * TSTEP;
            dst[i] = t < T ? __ldg(src + (size_t)t * (size_t)(npix >> 1)) : make_float4(0.f, 0.f, 0.f, 0.f);
        }
    };
    if ((long long)blockIdx.x < nblocks) load_block(blockIdx.x, wn);
    int dbuf = 0, in_buf = 0;                          // accumulator buffer in use, stages accumulated in it
    for (long long blk = blockIdx.x; blk < nblocks; blk += gridDim.x, ++it) {
        const int s = it & 1;
#pragma unroll
        for (int i = 0; i < ITEMS; ++i) w[i] = wn[i];
        if (blk + gridDim.x < nblocks) load_block(blk + gridDim.x, wn);
        if (pending[s]) { mbar_wait(mma_done + s, ph[s]); ph[s] ^= 1u; pending[s] = 0; }   // the MMAs that read this stage
        unsigned char* tile = base + (size_t)s * STAGE + (size_t)ktile * CT_TILE * (SPLIT ? 2 : 1);
#pragma unroll
        for (int i = 0; i < ITEMS; ++i) {
            const int t = t0 + i * TSTEP;
            if (t < T) {
                const int row = slice * TP + t;
                const uint32_t off = (uint32_t)(row >> 3) * 1024u + (uint32_t)(row & 7) * 128u + (uint32_t)((j16 ^ (row & 7)) << 4);
                const float4 x = w[i];
                const float4 hi = make_float4(to_tf32(x.x), to_tf32(x.y), to_tf32(x.z), to_tf32(x.w));
                *reinterpret_cast<float4*>(tile + off) = hi;
                if constexpr (SPLIT) {
                    const float4 lo = make_float4(to_tf32(x.x - hi.x), to_tf32(x.y - hi.y), to_tf32(x.z - hi.z), to_tf32(x.w - hi.w));
                    *reinterpret_cast<float4*>(tile + CT_TILE + off) = lo;
                }
            }
        }
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");     // the tensor core reads the tile through the async proxy
        asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
        __syncthreads();
        if (tid == 0) {
            asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
            const uint32_t sa0 = sbase + (uint32_t)s * STAGE;
            const uint32_t dst = tmem + (uint32_t)(dbuf * 128);
#pragma unroll
            for (int kt = 0; kt < TILES; ++kt)
#pragma unroll
                for (int k = 0; k < 4; ++k) {                  // K = 8 floats per instruction: 32 bytes further into the 128-byte rows
                    const uint32_t a0 = sa0 + (uint32_t)kt * CT_TILE * (SPLIT ? 2 : 1) + (uint32_t)k * 32u;
                    const uint64_t dh = ct_sdesc(a0);
                    umma_tf32(dst, dh, dh, idesc, (in_buf | kt | k) ? 1u : 0u);
                    if constexpr (SPLIT) {
                        const uint64_t dl = ct_sdesc(a0 + CT_TILE);
                        umma_tf32(dst, dh, dl, idesc, 1u);
                        umma_tf32(dst, dl, dh, idesc, 1u);
                    }
                }
            ct_commit(mma_done + s);
        }
        pending[s] = 1;
        if (++in_buf == drain_every) {
            // the MMAs of this stage are the last into buffer dbuf: wait for them (the next stage's go to the other buffer
            // and run under the drain), then add the buffer to the FP64 accumulators
            mbar_wait(mma_done + s, ph[s]); ph[s] ^= 1u; pending[s] = 0;
            drain(dbuf);
            dbuf ^= 1; in_buf = 0;
            __syncthreads();                                   // nobody overwrites the drained buffer's successor early
        }
    }
    for (int q = 0; q < 2; ++q) if (pending[q]) { mbar_wait(mma_done + q, ph[q]); ph[q] ^= 1u; pending[q] = 0; }
    if (in_buf) drain(dbuf);
    __syncthreads();
    // combine the S slices (fixed order) through shared memory and write this CTA's partial: [t][s'] lower triangle and all
    double* red = reinterpret_cast<double*>(base);           // [128 rows][TP] doubles = 64 KB at most
#pragma unroll
    for (int i = 0; i < NACC; ++i) red[(size_t)drow * TP + (warp >> 2) * NACC + i] = acc[i];
    __syncthreads();
    float2* out = partials + (size_t)blockIdx.x * T8 * T8;
    for (int e = tid; e < T * T; e += CT_THREADS) {
        const int t = e / T, s2 = e - t * T;
        double v = 0.0;
#pragma unroll
        for (int sl = 0; sl < S; ++sl) v += red[(size_t)(sl * TP + t) * TP + s2];
        out[t * T8 + s2] = make_float2((float)v, 0.f);
    }
    __syncthreads();
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "r"(256) : "memory");
}

// ------------------------------------------------------------------------------------------------
// The same single-pass TF32 Gram fed by TMA (the default single-pass form; holo_tune key 20 = 0 selects the kernel above).
// The register-fed kernel has ONE stage (64 KB per SM) of loads in flight and then waits for it: 4.0 TB/s.  Here the TMA unit writes the stack straight into the operand layout -- a 3-D box of
// [TP frames][S pieces][32 floats] with CU_TENSOR_MAP_SWIZZLE_128B lands as the 128 rows of a K-major SWIZZLE_128B tile, rows
// of frames t >= T zero-filled -- into a ring of CQ_NST stages, several stages ahead; the threads only round the landed values
// to TF32 IN PLACE (LDS.128, 4 x cvt.rna, STS.128 at the same address: no layout arithmetic, no bank conflicts), and the stage
// goes to the tensor core.  Row r = t S + sl of a tile holds piece sl of frame t: D = X X^T then carries the Gram of slice
// sl in the entries (t S + sl, t' S + sl), which the drain picks out of the TMEM columns.
// (2-D boxes of [TP frames][32 floats], which give slice-major rows, are request-rate bound at 4.07 TB/s with loads alone: the
// TMA unit fetches every 128-byte box row separately; in the 3-D box the S pieces of a frame are one contiguous run.  A raw
// landing ring with a second, converting copy into the operand layout moves 160 KB per 32 KB stage through the shared-memory
// port, which the MMAs -- A and B both read from shared memory, 128 B per clock while they run -- share: 72 / 605 us against
// 60 / 415 us for this form and 66.5 / 581 us for the register-fed kernel at 1024^2 x 32 / 2048^2 x 64.)
// ------------------------------------------------------------------------------------------------
constexpr int CQ_TILES = 2;                        // K-tiles per stage: 32 KB
constexpr int CQ_STAGE = CQ_TILES * CT_TILE;
constexpr int CQ_NST = 6;                          // ring stages: 192 KB, up to 4 in flight beside the one being rounded and the one in the MMAs
constexpr size_t CQ_SMEM = 1024 + (size_t)CQ_NST * CQ_STAGE + 256;

__device__ __forceinline__ void tma_3d_g2s(void* dst_smem, const CUtensorMap* tm, int c0, int c1, int c2, uint64_t* bar) {
    asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];"
                 ::"r"(smem_u32(dst_smem)), "l"(tm), "r"(c0), "r"(c1), "r"(c2), "r"(smem_u32(bar)) : "memory");
}

template <int TP>
__global__ void __launch_bounds__(CT_THREADS, 1)
k_cov_tf32_tma(const __grid_constant__ CUtensorMap tmH, float2* __restrict__ partials, long long npix, int T, int T8, int drain_every) {
    constexpr int S = 128 / TP;                       // pieces (K-slices) of a frame in the 128 rows of a tile
    constexpr int FPF = CQ_TILES * S * 32;            // floats of one frame per stage
    constexpr int PIX = FPF / 2;                      // pixels per stage
    extern __shared__ unsigned char smraw_[];
    const uint32_t s0 = smem_u32(smraw_);
    const uint32_t pad = (1024u - (s0 & 1023u)) & 1023u;
    unsigned char* base = smraw_ + pad;               // 1024-byte aligned stages
    const uint32_t sbase = s0 + pad;
    uint64_t* full = reinterpret_cast<uint64_t*>(base + (size_t)CQ_NST * CQ_STAGE);
    uint64_t* mma_done = full + CQ_NST;
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(mma_done + CQ_NST);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;

    if (tid == 0) {
        for (int i = 0; i < CQ_NST; ++i) { mbar_init(full + i, 1); mbar_init(mma_done + i, 1); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(tmem_slot)), "r"(256) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    pdl_wait();                                       // the holograms are complete (programmatic dependent launch)
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const uint32_t tmem = *tmem_slot;
    const uint32_t idesc = (1u << 4) | (2u << 7) | (2u << 10) | ((uint32_t)(128 >> 3) << 17) | ((uint32_t)(128 >> 4) << 24);
    const long long nblocks = npix / PIX;
    const long long first = blockIdx.x, step = gridDim.x;
    const long long niter = first < nblocks ? (nblocks - first + step - 1) / step : 0;

    // producer (thread 0): block `it` of this CTA -> stage it % NST: one box [TP frames][S pieces][32 floats] per K-tile
    auto issue = [&](long long it) {
        const int s = (int)(it % CQ_NST);
        const long long p0 = (first + it * step) * (CQ_TILES * S);  // first 32-float piece of the block inside a frame
        mbar_arrive_expect_tx(full + s, (uint32_t)CQ_STAGE);        // (zero-filled rows count as transferred bytes)
#pragma unroll
        for (int kt = 0; kt < CQ_TILES; ++kt)
            tma_3d_g2s(base + (size_t)s * CQ_STAGE + (size_t)kt * CT_TILE, &tmH, 0, (int)(p0 + kt * S), 0, full + s);
    };
    if (tid == 0)
        for (long long it = 0; it < niter && it < CQ_NST; ++it) issue(it);

    // FP64 accumulators: thread (row r = t S + sl, column half h) adds D[r][t' S + sl] for t' in [h TP/2, (h + 1) TP/2)
    constexpr int NACC = TP / 2;
    double acc[NACC];
#pragma unroll
    for (int i = 0; i < NACC; ++i) acc[i] = 0.0;
    const int drow = 32 * (warp & 3) + lane;
    const int dsl = drow % S, dh = warp >> 2;
    auto drain = [&](int buf) {
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
#pragma unroll
        for (int q = 0; q < 64 / 16; ++q) {            // the thread's half of the 128 columns, 16 at a time; it keeps the columns c = t' S + sl
            float v[16];
            tmem_ld16f(tmem + ((uint32_t)(32 * (warp & 3)) << 16) + (uint32_t)(buf * 128 + dh * 64 + 16 * q), v);
#pragma unroll
            for (int g = 0; g < 16 / S; ++g) {         // group g of S consecutive columns = one t'
                float x = v[g * S];
#pragma unroll
                for (int j = 1; j < S; ++j) x = dsl == j ? v[g * S + j] : x;
                acc[q * (16 / S) + g] += (double)x;
            }
        }
        asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    };

    int dbuf = 0, in_buf = 0;
    for (long long it = 0; it < niter; ++it) {
        const int s = (int)(it % CQ_NST);
        const uint32_t par = (uint32_t)((it / CQ_NST) & 1);
        mbar_wait(full + s, par);                                   // the stage has landed
        float4* st4 = reinterpret_cast<float4*>(base + (size_t)s * CQ_STAGE);
#pragma unroll
        for (int i = 0; i < CQ_STAGE / 16 / CT_THREADS; ++i) {      // round to nearest TF32, in place
            float4 x = st4[tid + i * CT_THREADS];
            x = make_float4(to_tf32(x.x), to_tf32(x.y), to_tf32(x.z), to_tf32(x.w));
            st4[tid + i * CT_THREADS] = x;
        }
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");     // the tensor core reads the tile through the async proxy
        asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
        __syncthreads();
        if (tid == 0) {
            asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
            const uint32_t sa0 = sbase + (uint32_t)s * CQ_STAGE;
            const uint32_t dst = tmem + (uint32_t)(dbuf * 128);
#pragma unroll
            for (int kt = 0; kt < CQ_TILES; ++kt)
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    const uint64_t dhh = ct_sdesc(sa0 + (uint32_t)kt * CT_TILE + (uint32_t)k * 32u);
                    umma_tf32(dst, dhh, dhh, idesc, (in_buf | kt | k) ? 1u : 0u);
                }
            ct_commit(mma_done + s);
            // refill the stage of the PREVIOUS iteration: its MMAs were issued a whole iteration ago
            if (it >= 1 && it - 1 + CQ_NST < niter) {
                const int sp = (int)((it - 1) % CQ_NST);
                mbar_wait(mma_done + sp, (uint32_t)(((it - 1) / CQ_NST) & 1));
                issue(it - 1 + CQ_NST);
            }
        }
        if (++in_buf == drain_every) {
            mbar_wait(mma_done + s, par);                           // the last MMAs into buffer dbuf (the next stage's go to the other one)
            drain(dbuf);
            dbuf ^= 1; in_buf = 0;
            __syncthreads();
        }
    }
    if (in_buf) {
        const long long it = niter - 1;
        mbar_wait(mma_done + (int)(it % CQ_NST), (uint32_t)((it / CQ_NST) & 1));   // commits complete in order: all MMAs are done
        drain(dbuf);
    }
    __syncthreads();
    // combine the S slices (fixed order) through shared memory: red[r = t S + sl][t'] and write this CTA's partial
    double* red = reinterpret_cast<double*>(base);           // [128 rows][TP] doubles (every stage has been consumed)
#pragma unroll
    for (int i = 0; i < NACC; ++i) red[(size_t)drow * TP + dh * NACC + i] = acc[i];
    __syncthreads();
    float2* out = partials + (size_t)blockIdx.x * T8 * T8;
    for (int e = tid; e < T * T; e += CT_THREADS) {
        const int t = e / T, s2 = e - t * T;
        double v = 0.0;
#pragma unroll
        for (int sl = 0; sl < S; ++sl) v += red[(size_t)(t * S + sl) * TP + s2];
        out[t * T8 + s2] = make_float2((float)v, 0.f);
    }
    __syncthreads();
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "r"(256) : "memory");
}

template <int TP, bool SPLIT>
int launch_tf32(holo_ctx* c, const float2* H, cudaStream_t st, int* nparts) {
    constexpr int TILES = SPLIT ? 2 : 4;
    constexpr int STAGE = TILES * CT_TILE * (SPLIT ? 2 : 1);
    constexpr int PIX = TILES * (128 / TP) * 32 / 2;
    constexpr size_t smem = 1024 + 2 * STAGE + 64;
    auto kern = k_cov_tf32<TP, SPLIT>;
    { const int rc = holo_ensure_smem_attr((const void*)kern, c->device, smem); if (rc) return rc; }
    const long long nblocks = c->npix / PIX;
    int grid = c->cov_grid_cap > 0 ? c->cov_grid_cap : c->num_sms;
    if (grid > c->cov_parts_cap) grid = c->cov_parts_cap;
    if ((long long)grid > nblocks) grid = (int)nblocks;
    int de = c->tune[HOLO_TUNE_COV_TF32_DRAIN];
    if (de < 1) de = 4;
    const int T8 = (c->T + 7) / 8 * 8;
    HoloProf prof(c, HOLO_K_COV_PARTIAL, st);
    kern<<<grid, CT_THREADS, smem, st>>>(H, c->cov_partials, c->npix, c->T, T8, de);
    HOLO_CUDA_OK(cudaGetLastError());
    *nparts = grid;
    return HOLO_OK;
}

// H viewed as a 3-D float tensor [2 npix / 32 pieces][T frames][32 floats] (dimension 0 = the 32 floats = 128 bytes of a piece,
// dimension 1 = the pieces of a frame, 128 bytes apart, dimension 2 = the frames); box = [TP frames][S pieces][32 floats], written
// with the 128-byte swizzle of the K-major operand layout; frames >= T are zero-filled
static int make_swizzled_map(CUtensorMap* tm, const float2* H, long long npix, int T, int TP) {
    static EncodeTiledFn encode = nullptr;
    if (!encode) {
        void* fn = nullptr;
        cudaDriverEntryPointQueryResult qres;
        HOLO_CUDA_OK(cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres));
        if (!fn || qres != cudaDriverEntryPointSuccess) { holo_set_error("cuTensorMapEncodeTiled not available"); return HOLO_ERR_CUDA; }
        encode = (EncodeTiledFn)fn;
    }
    const cuuint64_t gdim[3] = {32, (cuuint64_t)(2 * npix / 32), (cuuint64_t)T};
    const cuuint64_t gstr[2] = {128, (cuuint64_t)npix * sizeof(float2)};
    const cuuint32_t box[3] = {32, (cuuint32_t)(128 / TP), (cuuint32_t)TP};
    const cuuint32_t estr[3] = {1, 1, 1};
    const CUresult r = encode(tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, const_cast<float2*>(H), gdim, gstr, box, estr,
                              CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                              CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) { holo_set_error("cuTensorMapEncodeTiled (swizzled) failed (%d)", (int)r); return HOLO_ERR_CUDA; }
    return HOLO_OK;
}

template <int TP>
int launch_tf32_tma(holo_ctx* c, const float2* H, cudaStream_t st, int* nparts) {
    constexpr int PIX = CQ_TILES * (128 / TP) * 32 / 2;
    auto kern = k_cov_tf32_tma<TP>;
    { const int rc = holo_ensure_smem_attr((const void*)kern, c->device, CQ_SMEM); if (rc) return rc; }
    alignas(64) CUtensorMap tmH;
    { const int rc = make_swizzled_map(&tmH, H, c->npix, c->T, TP); if (rc) return rc; }
    const long long nblocks = c->npix / PIX;
    int grid = c->cov_grid_cap > 0 ? c->cov_grid_cap : c->num_sms;
    if (grid > c->cov_parts_cap) grid = c->cov_parts_cap;
    if ((long long)grid > nblocks) grid = (int)nblocks;
    int de = c->tune[HOLO_TUNE_COV_TF32_DRAIN];
    if (de < 1) de = 4;
    de *= 2;                                           // the key counts stages of four K-tiles; these stages hold two
    const int T8 = (c->T + 7) / 8 * 8;
    HoloProf prof(c, HOLO_K_COV_PARTIAL, st);
    HOLO_CUDA_OK(holo_launch_pdl(kern, dim3(grid), dim3(CT_THREADS), CQ_SMEM, st, tmH, c->cov_partials, c->npix, c->T, T8, de));
    *nparts = grid;
    return HOLO_OK;
}

}  // namespace

// Re C partials of the hologram stack on the tensor cores (tune key 13: 1 = TF32 with round-to-nearest conversion, 3 = 3 x TF32)
int holo_launch_cov_tf32(holo_ctx* c, const float2* H, float2* C, cudaStream_t st) {
    const bool split = c->tune[HOLO_TUNE_COV_TF32] == 3;
    if (c->npix % 256 != 0) { holo_set_error("the tensor-core Gram needs nx*ny to be a multiple of 256"); return HOLO_ERR_ARG; }
    int nparts = 0, rc;
    if (!split && c->tune[HOLO_TUNE_COV_TF32_TMA]) rc = c->T <= 32 ? launch_tf32_tma<32>(c, H, st, &nparts) : launch_tf32_tma<64>(c, H, st, &nparts);
    else if (c->T <= 32) rc = split ? launch_tf32<32, true>(c, H, st, &nparts) : launch_tf32<32, false>(c, H, st, &nparts);
    else            rc = split ? launch_tf32<64, true>(c, H, st, &nparts) : launch_tf32<64, false>(c, H, st, &nparts);
    if (rc) return rc;
    c->cov_nparts = nparts;
    return C ? holo_launch_cov_reduce(c, nparts, C, st) : HOLO_OK;
}
