// covariance.cu -- A3: C = H^{t*} H, C_ts = sum_p conj(H_t(p)) H_s(p)   (Eq. 4; R9)
//
// FP32 FFMA Gram of a tall-skinny matrix (N_p x T, T <= 64); FP32-ALU bound at T >= 32.
// The Hermitian lower half of C is cut into 8x8 complex blocks.  One warp owns either one off-diagonal
// block (64 complex accumulators) or a PAIR of diagonal blocks (2 x 36 entries, real diagonal): both cost
// 256 FFMA per pixel, so the eight consumer warps of a CTA (two per SM sub-partition) are exactly balanced
// and no redundant upper-triangle work is done.  The 32 lanes of a warp split the pixels of a staged
// chunk, so the only reduction is a once-per-CTA shuffle tree.  Warp 0 doubles as the producer: before
// each of its chunks it streams the chunk NS-2 ahead into a multi-stage shared-memory ring with 2-D TMA
// tensor copies (cp.async.bulk.tensor.2d + mbarrier complete_tx; one [8 rows x 128 pixels] box per row
// block -- 1-D bulk copies of single 1 KB rows were measured TMA-issue bound at 1.5 TB/s); rows t >= T of
// the last row block are zero-filled by the TMA unit (out-of-bounds fill).  The warps release a stage with
// one mbarrier arrive each: no __syncthreads and no per-thread copy loops in the steady state
// (256 threads, so every thread may hold the full 255 registers).
// Each CTA writes one partial; a second kernel sums the partials in a FIXED order in FP64
// (deterministic, bit-identical runs).  For T > 32 the blocks are split over gridDim.y CTA groups, each
// staging only the row blocks its jobs touch.
#include "holo_internal.cuh"
#include <string.h>
#include "tma.cuh"

#define COV_P 128            // pixels per stage (1 KB per row)
#define COV_NW 8             // consumer warps per CTA
#define COV_MAX_SLOTS 8      // row blocks (of 8 rows) staged per CTA group
#define COV_MAX_GROUPS 4
#define COV_MAX_STAGES 8
#define COV_SMEM_BUDGET (200 * 1024)

struct CovJob {              // one consumer warp
    int kind;                // 0 idle, 1 off-diagonal block (ra > rb), 2 pair of diagonal blocks (rb < 0: single)
    int sa, sb;              // stage slots of the two row blocks
    int ra, rb;              // global row-block indexes (output position)
};
struct CovGroup {
    int nslots, njobs;
    int rowblk[COV_MAX_SLOTS];
    CovJob job[COV_NW];
};
struct CovPlan {
    int ngroups;
    CovGroup g[COV_MAX_GROUPS];
};

__device__ __forceinline__ float warp_sum(float x) {
#pragma unroll
    for (int o = 16; o >= 1; o >>= 1) x += __shfl_xor_sync(0xffffffffu, x, o);
    return x;
}

// An accumulator is the pair (re, im).  (The packed fma.rn.f32x2 form of these updates was measured 16 % slower here:
// the operand-pair moves land on the FMA pipe.)
typedef float2 pair_t;
__device__ __forceinline__ pair_t pack2(float lo, float hi) { return make_float2(lo, hi); }
__device__ __forceinline__ void unpack2(pair_t v, float& lo, float& hi) { lo = v.x; hi = v.y; }
__device__ __forceinline__ void ffma2(pair_t& acc, pair_t a, pair_t b) { acc.x = fmaf(a.x, b.x, acc.x); acc.y = fmaf(a.y, b.y, acc.y); }
__device__ __forceinline__ pair_t pzero() { return make_float2(0.f, 0.f); }

// partials layout: [part][T8][T8] float2 (T8 = T rounded up to 8), only entries s <= t are written
__global__ void __launch_bounds__(COV_NW * 32, 1)
k_cov_partial(const __grid_constant__ CUtensorMap tmH, float2* __restrict__ partials, long long npix, int T, int T8,
              int nstages, const CovPlan plan) {
    extern __shared__ __align__(128) unsigned char smraw[];
    uint64_t* full = reinterpret_cast<uint64_t*>(smraw);
    uint64_t* empty = full + COV_MAX_STAGES;
    float2* ring = reinterpret_cast<float2*>(smraw + 128);
    const CovGroup& g = plan.g[blockIdx.y];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int nslots = g.nslots;
    const int stage_elems = nslots * 8 * COV_P;
    const long long nchunks = npix / COV_P;

    if (tid == 0) {
        for (int s = 0; s < nstages; ++s) { mbar_init(full + s, 1); mbar_init(empty + s, (uint32_t)g.njobs); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    // ---------------------------------------------------- producer state (used by warp 0 only)
    int ps = 0; uint32_t pph = 0;
    long long pchunk = blockIdx.x;
    auto issue = [&]() {
        if (pchunk >= nchunks) return;
        mbar_wait(empty + ps, pph ^ 1u);
        if (lane == 0) mbar_arrive_expect_tx(full + ps, (uint32_t)stage_elems * (uint32_t)sizeof(float2));
        __syncwarp();
        if (lane < nslots)      // one [8 rows x COV_P pixels] box per row block; coordinates in floats / rows
            tma_2d_g2s(ring + (size_t)ps * stage_elems + lane * 8 * COV_P, &tmH, (int)(pchunk * (2 * COV_P)), 8 * g.rowblk[lane], full + ps);
        pchunk += gridDim.x;
        if (++ps == nstages) { ps = 0; pph ^= 1u; }
    };
    if (warp == 0)
        for (int d = 0; d < nstages - 2; ++d) issue();
    // ---------------------------------------------------- consumer warps
    // One pixel per lane per trip: 16 LDS.64 + 256 FFMA, a 4.5 KB loop body.  An accumulator is the pair
    // (re, im);  acc += conj(a) b  =  (ax,ax)*(bx,by) + (ay,-ay)*(by,bx)  (pair_t / ffma2 below).
    // Measured alternative (profiles/r01c.md): two pixels per trip with LDS.128 (same speed, twice the code).
    const CovJob job = g.job[warp];      // make_plan orders the jobs so that one SM sub-partition (warp & 3) runs one kind
    if (job.kind == 0) return;
    float2* out = partials + (size_t)blockIdx.x * T8 * T8;
    int s = 0; uint32_t ph = 0;
    if (job.kind == 1) {
        pair_t acc[8][8];
#pragma unroll
        for (int i = 0; i < 8; ++i)
#pragma unroll
            for (int j = 0; j < 8; ++j) acc[i][j] = pzero();
        for (long long chunk = blockIdx.x; chunk < nchunks; chunk += gridDim.x) {
            if (warp == 0) issue();
            mbar_wait(full + s, ph);
            const float2* A = ring + (size_t)s * stage_elems + job.sa * 8 * COV_P + lane;
            const float2* B = ring + (size_t)s * stage_elems + job.sb * 8 * COV_P + lane;
#pragma unroll 1
            for (int it = 0; it < COV_P / 32; ++it) {
                pair_t a1[8], a2[8], b1[8], b2[8];
#pragma unroll
                for (int i = 0; i < 8; ++i) { const float2 a = A[i * COV_P + it * 32]; a1[i] = pack2(a.x, a.x); a2[i] = pack2(a.y, -a.y); }
#pragma unroll
                for (int j = 0; j < 8; ++j) { const float2 b = B[j * COV_P + it * 32]; b1[j] = pack2(b.x, b.y); b2[j] = pack2(b.y, b.x); }
#pragma unroll
                for (int i = 0; i < 8; ++i)
#pragma unroll
                    for (int j = 0; j < 8; ++j) { ffma2(acc[i][j], a1[i], b1[j]); ffma2(acc[i][j], a2[i], b2[j]); }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(empty + s);
            if (++s == nstages) { s = 0; ph ^= 1u; }
        }
#pragma unroll
        for (int i = 0; i < 8; ++i)
#pragma unroll
            for (int j = 0; j < 8; ++j) {
                float x, y;
                unpack2(acc[i][j], x, y);
                x = warp_sum(x); y = warp_sum(y);
                if (lane == 0) out[(job.ra * 8 + i) * T8 + (job.rb * 8 + j)] = make_float2(x, y);
            }
    } else {
        // two diagonal blocks: entries i > j complex; i == j real, accumulated as the pair (sum ax^2, sum ay^2)
        pair_t lo[2][28], dg[2][8];
#pragma unroll
        for (int d = 0; d < 2; ++d) {
#pragma unroll
            for (int e = 0; e < 28; ++e) lo[d][e] = pzero();
#pragma unroll
            for (int i = 0; i < 8; ++i) dg[d][i] = pzero();
        }
        const bool two = job.rb >= 0;
        for (long long chunk = blockIdx.x; chunk < nchunks; chunk += gridDim.x) {
            if (warp == 0) issue();
            mbar_wait(full + s, ph);
            const float2* A0 = ring + (size_t)s * stage_elems + job.sa * 8 * COV_P + lane;
            const float2* A1 = ring + (size_t)s * stage_elems + job.sb * 8 * COV_P + lane;
#pragma unroll 1
            for (int it = 0; it < COV_P / 32; ++it) {
#pragma unroll
                for (int d = 0; d < 2; ++d) {
                    if (d == 1 && !two) continue;
                    const float2* A = d == 0 ? A0 : A1;
                    pair_t a1[8], a2[8], b1[8], b2[8];
#pragma unroll
                    for (int i = 0; i < 8; ++i) {
                        const float2 a = A[i * COV_P + it * 32];
                        a1[i] = pack2(a.x, a.x); a2[i] = pack2(a.y, -a.y); b1[i] = pack2(a.x, a.y); b2[i] = pack2(a.y, a.x);
                    }
#pragma unroll
                    for (int i = 0; i < 8; ++i) {
                        ffma2(dg[d][i], b1[i], b1[i]);
#pragma unroll
                        for (int j = 0; j < i; ++j) { ffma2(lo[d][i * (i - 1) / 2 + j], a1[i], b1[j]); ffma2(lo[d][i * (i - 1) / 2 + j], a2[i], b2[j]); }
                    }
                }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(empty + s);
            if (++s == nstages) { s = 0; ph ^= 1u; }
        }
#pragma unroll
        for (int d = 0; d < 2; ++d) {
            if (d == 1 && !two) continue;
            const int r = (d == 0 ? job.ra : job.rb) * 8;
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                float x, y;
                unpack2(dg[d][i], x, y);
                x = warp_sum(x + y);
                if (lane == 0) out[(r + i) * T8 + (r + i)] = make_float2(x, 0.f);
#pragma unroll
                for (int j = 0; j < i; ++j) {
                    unpack2(lo[d][i * (i - 1) / 2 + j], x, y);
                    x = warp_sum(x); y = warp_sum(y);
                    if (lane == 0) out[(r + i) * T8 + (r + j)] = make_float2(x, y);
                }
            }
        }
    }
}

struct RealJob { int kind, a16, b8; };        // kind 0: rows [16 a16, +16) x rows [8 b8, +8);  kind 1: lower triangle of rows [16 a16, +16)
struct RealPlan { int njobs[2]; RealJob job[2][COV_NW]; };

// ------------------------------------------------------------------------------------------------
// Real part only, for the hologram stacks of holo_process / holo_submit.  There H_t = F[q d_t] with d_t
// real, q unimodular and F unitary up to nx ny, so C_ts = nx ny sum_x d_t d_s is REAL in exact arithmetic
// (R8, R21): the imaginary part the complex kernel would compute is rounding noise and half the
// FFMA work.  Re C_ts = sum_p (re_t re_s + im_t im_s): a real Gram over 2 N_p samples.  Jobs (one real
// accumulator per entry): "off" = rows [16,32) x one 8-row block of [0,16) (128 entries, 24 loads per pixel),
// "diag16" = lower triangle of a 16-row block (136 entries, 16 loads).  Four jobs cover T <= 32; warps w and
// w+4 run the same job on alternate 128-pixel chunks (two partials per CTA).  T <= 16: one diag16 job,
// four warps take every fourth chunk each.  32 < T <= 64: nine or sixteen jobs over two CTA groups (gridDim.y),
// every CTA stages all T rows.  Same TMA ring / mbarrier protocol as k_cov_partial.
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(COV_NW * 32, 1)
k_cov_partial_real(const __grid_constant__ CUtensorMap tmH, float2* __restrict__ partials, long long npix, int T8,
                   int nstages, int nslots, int ngroups, int ahead, const RealPlan plan, int rb0, int nrb) {
    extern __shared__ __align__(128) unsigned char smraw[];
    uint64_t* full = reinterpret_cast<uint64_t*>(smraw);
    uint64_t* empty = full + COV_MAX_STAGES;
    float2* ring = reinterpret_cast<float2*>(smraw + 128);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int stage_elems = nslots * 8 * COV_P;
    const long long nchunks = npix / COV_P;
    // ngroups warp groups: group g owns the CTA's chunks k = g (mod ngroups); the jobs come from plan.job[blockIdx.y]
    const int njobs = plan.njobs[blockIdx.y];
    const int nactive = njobs * ngroups;                 // <= 8 warps
    if (tid == 0) {
        for (int s = 0; s < nstages; ++s) { mbar_init(full + s, 1); mbar_init(empty + s, (uint32_t)njobs); }   // nstages is a multiple of ngroups: a stage always serves the same group
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    pdl_trigger();                                        // (k_cov_reduce)
    pdl_wait();                                           // the holograms are complete
    __syncthreads();
    int ps = 0; uint32_t pph = 0;
    long long pchunk = blockIdx.x;
    auto issue = [&]() {
        if (pchunk >= nchunks) return;
        mbar_wait(empty + ps, pph ^ 1u);
        if (lane == 0) mbar_arrive_expect_tx(full + ps, (uint32_t)stage_elems * (uint32_t)sizeof(float2));
        __syncwarp();
        // nrb != 0: the T rows are a window of a ring of nrb 8-row blocks that starts at block rb0 (holo_push)
        if (lane < nslots) tma_2d_g2s(ring + (size_t)ps * stage_elems + lane * 8 * COV_P, &tmH, (int)(pchunk * (2 * COV_P)),
                                      8 * (nrb ? (rb0 + lane) % nrb : lane), full + ps);
        pchunk += gridDim.x;
        if (++ps == nstages) { ps = 0; pph ^= 1u; }
    };
    if (warp == 0)
        for (int d = 0; d < ahead; ++d) issue();
    if (warp >= nactive) return;
    const int group = warp / njobs;
    const RealJob job = plan.job[blockIdx.y][warp % njobs];
    float2* out = partials + ((size_t)blockIdx.x * ngroups + group) * T8 * T8;
    int s = 0; uint32_t ph = 0;
    if (job.kind == 0) {
        float acc[16][8];
#pragma unroll
        for (int i = 0; i < 16; ++i)
#pragma unroll
            for (int j = 0; j < 8; ++j) acc[i][j] = 0.f;
        int k = 0;
        for (long long chunk = blockIdx.x; chunk < nchunks; chunk += gridDim.x, ++k) {
            if (warp == 0) issue();
            if (k % ngroups != group) { if (++s == nstages) { s = 0; ph ^= 1u; } continue; }
            mbar_wait(full + s, ph);
            const float2* A = ring + (size_t)s * stage_elems + job.a16 * 16 * COV_P + lane;
            const float2* B = ring + (size_t)s * stage_elems + job.b8 * 8 * COV_P + lane;
#pragma unroll 1
            for (int it = 0; it < COV_P / 32; ++it) {
                float2 a[16], b[8];
#pragma unroll
                for (int i = 0; i < 16; ++i) a[i] = A[i * COV_P + it * 32];
#pragma unroll
                for (int j = 0; j < 8; ++j) b[j] = B[j * COV_P + it * 32];
#pragma unroll
                for (int i = 0; i < 16; ++i)
#pragma unroll
                    for (int j = 0; j < 8; ++j) acc[i][j] = fmaf(a[i].y, b[j].y, fmaf(a[i].x, b[j].x, acc[i][j]));
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(empty + s);
            if (++s == nstages) { s = 0; ph ^= 1u; }
        }
#pragma unroll
        for (int i = 0; i < 16; ++i)
#pragma unroll
            for (int j = 0; j < 8; ++j) {
                const float x = warp_sum(acc[i][j]);
                if (lane == 0 && job.a16 * 16 + i < T8) out[(job.a16 * 16 + i) * T8 + (job.b8 * 8 + j)] = make_float2(x, 0.f);
            }
    } else {
        const int r0 = job.a16 * 16;
        float acc[136];
#pragma unroll
        for (int e = 0; e < 136; ++e) acc[e] = 0.f;
        int k = 0;
        for (long long chunk = blockIdx.x; chunk < nchunks; chunk += gridDim.x, ++k) {
            if (warp == 0) issue();
            if (k % ngroups != group) { if (++s == nstages) { s = 0; ph ^= 1u; } continue; }
            mbar_wait(full + s, ph);
            const float2* A = ring + (size_t)s * stage_elems + r0 * COV_P + lane;
#pragma unroll 1
            for (int it = 0; it < COV_P / 32; ++it) {
                float2 a[16];
#pragma unroll
                for (int i = 0; i < 16; ++i) a[i] = A[i * COV_P + it * 32];
#pragma unroll
                for (int i = 0; i < 16; ++i)
#pragma unroll
                    for (int j = 0; j <= i; ++j) acc[i * (i + 1) / 2 + j] = fmaf(a[i].y, a[j].y, fmaf(a[i].x, a[j].x, acc[i * (i + 1) / 2 + j]));
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(empty + s);
            if (++s == nstages) { s = 0; ph ^= 1u; }
        }
#pragma unroll
        for (int i = 0; i < 16; ++i)
#pragma unroll
            for (int j = 0; j <= i; ++j) {
                const float x = warp_sum(acc[i * (i + 1) / 2 + j]);
                if (lane == 0 && r0 + i < T8) out[(r0 + i) * T8 + (r0 + j)] = make_float2(x, 0.f);
            }
    }
}

// fixed-order FP64 reduction over the partials: one warp per lower-triangle entry, lane l sums parts
// l, l+32, ... in order, then a fixed shuffle tree (deterministic).  Writes the full Hermitian C (both
// triangles), diagonal imaginary parts forced to 0.
// Cd != nullptr: the FP64 sums are also kept ([T][T] double2, both triangles) for the centring step of holo_push
__global__ void __launch_bounds__(256) k_cov_reduce(const float2* __restrict__ partials, int nparts, int T, int T8, float2* __restrict__ C,
                                                    double2* __restrict__ Cd) {
    const int w = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
    pdl_trigger();                                        // (the single-CTA eigensolver)
    pdl_wait();
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
        if (Cd) { Cd[t * T + s] = make_double2(re, s == t ? 0.0 : im); Cd[s * T + t] = make_double2(re, s == t ? 0.0 : -im); }
    }
}

// Sliding-window form (holo_push): the ring holds G_t = F[q (I_t - m0)] for a FIXED reference image m0, and the
// holograms of the current window are H_t = G_t - mean_t G.  Their covariance is C = J Gamma J with Gamma = G^H G and
// J = I - 11^T/T:  C_ts = Gamma_ts - rho_t/T - conj(rho_s)/T + tau/T^2  (rho = row sums, tau = total), done in
// FP64 on the unrounded sums of the reduction.  One CTA.
// Gs != nullptr: slot-indexed FP64 store of the (real) Gram of the hologram ring, Gs[slot_t * Rn + slot_s]; the window
// is slots a0 .. a0+T-1 (mod Rn).  scatter = 1: Gd (a full recomputation) is also copied into Gs; scatter = 0: Gd is not
// used, the window is gathered from Gs (incremental update: only the new rows / columns were recomputed).
__global__ void __launch_bounds__(256) k_center_gram(const double2* __restrict__ Gd, int T, float2* __restrict__ C,
                                                     double* __restrict__ Gs, int Rn, int a0, int scatter) {
    __shared__ double2 rho[HOLO_MAX_T];
    __shared__ double2 tau;
    const bool gather = Gs && !scatter;
    auto slot = [&](int t) { return (a0 + t) % Rn; };
    auto get = [&](int t, int s) { return gather ? make_double2(Gs[slot(t) * Rn + slot(s)], 0.0) : Gd[t * T + s]; };
    if (Gs && scatter)
        for (int i = threadIdx.x; i < T * T; i += blockDim.x) { const int t = i / T, s = i - t * T; Gs[slot(t) * Rn + slot(s)] = Gd[i].x; }
    if (Gs && scatter) __syncthreads();
    for (int t = threadIdx.x >> 5; t < T; t += blockDim.x >> 5) {         // one warp per row, fixed summation order
        double2 r = make_double2(0.0, 0.0);
        for (int s = threadIdx.x & 31; s < T; s += 32) { const double2 g = get(t, s); r.x += g.x; r.y += g.y; }
#pragma unroll
        for (int o = 16; o >= 1; o >>= 1) { r.x += __shfl_xor_sync(0xffffffffu, r.x, o); r.y += __shfl_xor_sync(0xffffffffu, r.y, o); }
        if ((threadIdx.x & 31) == 0) rho[t] = r;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        double2 acc = make_double2(0.0, 0.0);
        for (int t = 0; t < T; ++t) { acc.x += rho[t].x; acc.y += rho[t].y; }
        tau = acc;
    }
    __syncthreads();
    const double iT = 1.0 / (double)T;
    for (int i = threadIdx.x; i < T * T; i += blockDim.x) {
        const int t = i / T, s = i - t * T;
        const double2 g = get(t, s);
        const double re = g.x - (rho[t].x + rho[s].x) * iT + tau.x * iT * iT;
        const double im = g.y - (rho[t].y - rho[s].y) * iT;               // tau is real for a Hermitian Gamma
        C[i] = make_float2((float)re, t == s ? 0.f : (float)im);
    }
}

// incremental update: FP64 sums of the partial entries (row r, new column cn) -> Gs, both orientations.
// grid = (T rows, newb blocks), 8 warps: warp j of the CTA takes column j of the block, lanes split the parts.
__global__ void __launch_bounds__(256) k_cov_reduce_new(const float2* __restrict__ partials, int nparts, int T, int T8, int newb,
                                                        double* __restrict__ Gs, int Rn, int a0) {
    const int lane = threadIdx.x & 31, j = threadIdx.x >> 5;
    const int r = blockIdx.x, cn = T8 - 8 * newb + 8 * blockIdx.y + j;
    if (cn >= T) return;
    const float2* p = partials + r * T8 + cn;
    double re = 0.0;
    for (int k = lane; k < nparts; k += 32) re += (double)p[(size_t)k * T8 * T8].x;
#pragma unroll
    for (int o = 16; o >= 1; o >>= 1) re += __shfl_xor_sync(0xffffffffu, re, o);
    if (lane == 0) {
        const int sr = (a0 + r) % Rn, sc = (a0 + cn) % Rn;
        Gs[sr * Rn + sc] = re;
        Gs[sc * Rn + sr] = re;
    }
}

// ---- host: split the block lower triangle into CTA groups of <= COV_NW warp jobs
static int slot_of(CovGroup& g, int rb) {
    for (int k = 0; k < g.nslots; ++k) if (g.rowblk[k] == rb) return k;
    g.rowblk[g.nslots] = rb;
    return g.nslots++;
}
static void add_off(CovGroup& g, int bi, int bj) {
    CovJob& j = g.job[g.njobs++];
    j.kind = 1; j.ra = bi; j.rb = bj; j.sa = slot_of(g, bi); j.sb = slot_of(g, bj);
}
static void add_diag(CovGroup& g, int b0, int b1) {
    CovJob& j = g.job[g.njobs++];
    j.kind = 2; j.ra = b0; j.rb = b1; j.sa = slot_of(g, b0); j.sb = b1 >= 0 ? slot_of(g, b1) : 0;
}
// all jobs inside the row-block range [lo, hi) (hi - lo <= 4): <= 6 off-diagonal + 2 diagonal pairs
static void add_triangle(CovGroup& g, int lo, int hi) {
    for (int bi = lo; bi < hi; ++bi)
        for (int bj = lo; bj < bi; ++bj) add_off(g, bi, bj);
    for (int b = lo; b < hi; b += 2) add_diag(g, b, b + 1 < hi ? b + 1 : -1);
}
// warps w and w+4 share an SM sub-partition: put the diagonal-pair jobs on sub-partition 3 so that every
// sub-partition runs a single loop body (instruction-cache footprint)
static void order_jobs(CovGroup& g) {
    CovJob off[COV_NW], dia[COV_NW];
    int no = 0, nd = 0;
    for (int k = 0; k < g.njobs; ++k) (g.job[k].kind == 1 ? off[no++] : dia[nd++]) = g.job[k];
    int io = 0, id = 0;
    for (int w = 0; w < g.njobs; ++w) {
        const bool want_diag = (w & 3) == 3 || io == no;
        g.job[w] = (want_diag && id < nd) ? dia[id++] : off[io++];
    }
}
static void make_plan_groups(int nb, CovPlan* p);
static void make_plan(int nb, CovPlan* p) {
    make_plan_groups(nb, p);
    for (int k = 0; k < p->ngroups; ++k) order_jobs(p->g[k]);
}
static void make_plan_groups(int nb, CovPlan* p) {
    memset(p, 0, sizeof(*p));
    if (nb <= 4) { p->ngroups = 1; add_triangle(p->g[0], 0, nb); return; }
    // nb in 5..8: A = [0,4), B = [4,nb): triangle(A), triangle(B), rectangle B x A in strips of two block rows
    add_triangle(p->g[0], 0, 4);
    add_triangle(p->g[1], 4, nb);
    p->ngroups = 2;
    for (int b0 = 4; b0 < nb; b0 += 2) {
        CovGroup& g = p->g[p->ngroups++];
        for (int bi = b0; bi < b0 + 2 && bi < nb; ++bi)
            for (int bj = 0; bj < 4; ++bj) add_off(g, bi, bj);
    }
}

static int launch_cov_real(holo_ctx* c, const float2* H, float2* C, cudaStream_t st) {
    const int T = c->T, T8 = (T + 7) / 8 * 8, nb16 = (T8 + 15) / 16;
    // jobs: one diag16 per 16-row block, two [16 x 8] rectangles per pair of 16-row blocks
    RealPlan plan;
    memset(&plan, 0, sizeof(plan));
    RealJob all[16];
    int n = 0;
    const int newb = c->cov_new_blocks;                    // holo_push: only the products with the newest 8-row blocks
    if (newb > 0) {
        for (int b = T8 / 8 - newb; b < T8 / 8; ++b)
            for (int a = 0; a < nb16; ++a) all[n++] = RealJob{0, a, b};     // all rows x new block (upper-triangle entries too)
    } else {
        for (int a = 1; a < nb16; ++a)
            for (int b = 0; b < a; ++b) { all[n++] = RealJob{0, a, 2 * b}; all[n++] = RealJob{0, a, 2 * b + 1}; }
        for (int a = 0; a < nb16; ++a) all[n++] = RealJob{1, a, 0};
    }
    const int gy = n > COV_NW ? 2 : 1;
    for (int k = 0; k < n; ++k) { const int g = gy == 2 ? (k & 1) : 0; plan.job[g][plan.njobs[g]++] = all[k]; }
    const int ngroups = n == 4 ? 2 : n == 2 ? 4 : n == 1 ? 4 : 1;       // spare warps take alternate chunks
    const int nslots = nb16 * 2;
    const size_t stage_bytes = (size_t)nslots * 8 * COV_P * sizeof(float2);
    int nstages = (int)(COV_SMEM_BUDGET / stage_bytes);
    if (nstages > COV_MAX_STAGES) nstages = COV_MAX_STAGES;
    nstages -= nstages % ngroups;                          // a stage always serves the same warp group
    const int ahead = nstages > 3 ? nstages - 2 : nstages - 1;
    const size_t smem = 128 + (size_t)nstages * stage_bytes;
    { const int rc = holo_ensure_smem_attr((const void*)k_cov_partial_real, c->device, COV_SMEM_BUDGET + 128); if (rc) return rc; }
    const long long nchunks = c->npix / COV_P;
    int gx = (c->cov_grid_cap > 0 ? c->cov_grid_cap : c->tune[HOLO_TUNE_COV_GRIDX]) / gy;   // all CTAs co-resident: one per SM
    if (gx < 1) gx = 1;
    if (gx * ngroups > c->cov_parts_cap) gx = c->cov_parts_cap / ngroups;
    if ((long long)gx > nchunks) gx = (int)nchunks;
    alignas(64) CUtensorMap tmH;
    { const int rc = holo_make_tensor_map(&tmH, H, c->npix, c->ring_nrb ? 8 * c->ring_nrb : T, COV_P); if (rc) return rc; }
    {
        HoloProf prof(c, HOLO_K_COV_PARTIAL, st);
        HOLO_CUDA_OK(holo_launch_pdl(k_cov_partial_real, dim3(gx, gy), dim3(COV_NW * 32), smem, st, tmH, c->cov_partials, c->npix, T8, nstages, nslots,
                                     ngroups, ahead, plan, c->ring_rb0, c->ring_nrb));
    }
    HOLO_CUDA_OK(cudaGetLastError());
    c->cov_nparts = gx * ngroups;
    if (newb > 0) {
        // new rows / columns -> slot-indexed FP64 store, then gather + centre the window
        const int Rn = 8 * c->ring_nrb, a0 = 8 * c->ring_rb0;
        HoloProf prof(c, HOLO_K_COV_REDUCE, st);
        k_cov_reduce_new<<<dim3(T, newb), 256, 0, st>>>(c->cov_partials, c->cov_nparts, T, T8, newb, c->Gs, Rn, a0);
        HOLO_CUDA_OK(cudaGetLastError());
        k_center_gram<<<1, 256, 0, st>>>(nullptr, T, C, c->Gs, Rn, a0, 0);
        HOLO_CUDA_OK(cudaGetLastError());
        return HOLO_OK;
    }
    return C ? holo_launch_cov_reduce(c, c->cov_nparts, C, st) : HOLO_OK;
}

int holo_launch_cov_reduce(holo_ctx* c, int nparts, float2* C, cudaStream_t st) {
    const int T = c->T, T8 = (T + 7) / 8 * 8, n = T * T;
    HoloProf prof(c, HOLO_K_COV_REDUCE, st);
    HOLO_CUDA_OK(holo_launch_pdl(k_cov_reduce, dim3((n * 32 + 255) / 256), dim3(256), 0, st, (const float2*)c->cov_partials, nparts, T, T8, C,
                                 c->center_gram ? c->Cd : (double2*)nullptr));
    HOLO_CUDA_OK(cudaGetLastError());
    if (c->center_gram) {                                  // holo_push: C <- J Gamma J
        k_center_gram<<<1, 256, 0, st>>>(c->Cd, T, C, c->ring_nrb ? c->Gs : nullptr, 8 * c->ring_nrb, 8 * c->ring_rb0, 1);
        HOLO_CUDA_OK(cudaGetLastError());
    }
    return HOLO_OK;
}

// real_only: the caller guarantees that C is real in exact arithmetic (holograms produced by holo_fresnel)
int holo_launch_covariance(holo_ctx* c, const float2* H, float2* C, cudaStream_t st, bool real_only) {
    const int T = c->T, T8 = (T + 7) / 8 * 8, nb = T8 / 8;
    if (nb < 1 || nb > 8) { holo_set_error("T out of range"); return HOLO_ERR_ARG; }
    if (real_only && c->tune[HOLO_TUNE_COV_REAL] && c->tune[HOLO_TUNE_COV_TF32] && !c->center_gram && !c->cov_new_blocks && !c->ring_nrb)
        return holo_launch_cov_tf32(c, H, C, st);
    if (real_only && c->tune[HOLO_TUNE_COV_REAL]) return launch_cov_real(c, H, C, st);
    CovPlan plan;
    make_plan(nb, &plan);
    int max_slots = 0;
    for (int k = 0; k < plan.ngroups; ++k) max_slots = plan.g[k].nslots > max_slots ? plan.g[k].nslots : max_slots;
    const size_t stage_bytes = (size_t)max_slots * 8 * COV_P * sizeof(float2);
    int nstages = (int)(COV_SMEM_BUDGET / stage_bytes);
    if (nstages > COV_MAX_STAGES) nstages = COV_MAX_STAGES;
    if (nstages < 3) { holo_set_error("covariance stage ring does not fit"); return HOLO_ERR_STATE; }
    const size_t smem = 128 + (size_t)nstages * stage_bytes;
    { const int rc = holo_ensure_smem_attr((const void*)k_cov_partial, c->device, COV_SMEM_BUDGET + 128); if (rc) return rc; }
    const long long nchunks = c->npix / COV_P;
    int gx = c->tune[HOLO_TUNE_COV_GRIDX] / plan.ngroups;          // all CTAs co-resident: one per SM
    if (gx < 1) gx = 1;
    if (gx > c->cov_parts_cap) gx = c->cov_parts_cap;
    if ((long long)gx > nchunks) gx = (int)nchunks;
    alignas(64) CUtensorMap tmH;
    { const int rc = holo_make_tensor_map(&tmH, H, c->npix, T, COV_P); if (rc) return rc; }
    {
        HoloProf prof(c, HOLO_K_COV_PARTIAL, st);
        k_cov_partial<<<dim3(gx, plan.ngroups), COV_NW * 32, smem, st>>>(tmH, c->cov_partials, c->npix, T, T8, nstages, plan);
    }
    HOLO_CUDA_OK(cudaGetLastError());
    c->cov_nparts = gx;
    return C ? holo_launch_cov_reduce(c, c->cov_nparts, C, st) : HOLO_OK;
}
