// project.cu -- A5 + A6 fused:  M(p) = sum_{k in S} | sum_t H_t(p) V_{t,k} |^2     (Eq. 6-7)
// Reads the hologram stack once, never stores P.  Two exact forms (R12):
//   direct     : sum over the columns k in S = [k_lo,k_hi]
//   complement : (V unitary) deflation  H'_t = H_t - sum_{k not in S} P_k conj(V_tk),  M = sum_t |H'_t|^2,
//                used when the complement of S is smaller than S.  Algebraically equal to
//                sum_t|H_t|^2 - sum_{k not in S}|P_k|^2, but without the catastrophic cancellation of that
//                subtraction when the rejected clutter carries almost all of the energy (the method's use case).
// The same kernel serves the Fourier demodulation of Eq. 8-9 with V := W.
#include "holo_internal.cuh"
#include "tma.cuh"

struct ProjArgs {
    const float2* H;
    const float2* V;       // [T][T] row-major, column = component
    float* M;
    long long npix;
    int T;
    int r0_lo, r0_hi;      // first 0-based inclusive column range (empty if lo > hi)
    int r1_lo, r1_hi;      // second range
    int complement;        // 1: deflation form (the ranges are the REJECTED components); always taken by the k_project_deflate* kernels
    int center;            // 1: subtract the per-pixel mean over t first (sliding-window form: H_t = G_t - mean_t G)
};

template <int NC, int PIX>      // PIX = pixels per thread (2: float4 loads; 1 for very wide component sets)
__global__ void __launch_bounds__(256) k_project(const ProjArgs a) {
    __shared__ __align__(16) float2 Vs[HOLO_MAX_T * NC];          // [t][c], zero padded
    const int tid = threadIdx.x;
    const int n0 = a.r0_hi - a.r0_lo + 1 > 0 ? a.r0_hi - a.r0_lo + 1 : 0;
    for (int i = tid; i < a.T * NC; i += blockDim.x) {
        const int t = i / NC, c = i - t * NC;
        int col = -1;
        if (c < n0) col = a.r0_lo + c;
        else if (c - n0 <= a.r1_hi - a.r1_lo) col = a.r1_lo + (c - n0);
        Vs[i] = col >= 0 ? a.V[t * a.T + col] : make_float2(0.f, 0.f);
    }
    __syncthreads();
    const long long item = (long long)blockIdx.x * blockDim.x + tid;     // PIX adjacent pixels per thread
    if (item * PIX >= a.npix) return;
    const long long fstride = a.npix / PIX;
    float2 acc[PIX][NC];
#pragma unroll
    for (int x = 0; x < PIX; ++x)
#pragma unroll
        for (int c = 0; c < NC; ++c) acc[x][c] = make_float2(0.f, 0.f);
#pragma unroll 4
    for (int t = 0; t < a.T; ++t) {
        float2 h[PIX];
        if constexpr (PIX == 2) {
            const float4 w = __ldg(reinterpret_cast<const float4*>(a.H) + item + (long long)t * fstride);
            h[0] = make_float2(w.x, w.y); h[1] = make_float2(w.z, w.w);
        } else {
            h[0] = __ldg(a.H + item + (long long)t * fstride);
        }
#pragma unroll
        for (int c = 0; c < NC; ++c) {
            const float2 v = Vs[t * NC + c];
#pragma unroll
            for (int x = 0; x < PIX; ++x) {
                acc[x][c].x = fmaf(h[x].x, v.x, fmaf(-h[x].y, v.y, acc[x][c].x));
                acc[x][c].y = fmaf(h[x].x, v.y, fmaf(h[x].y, v.x, acc[x][c].y));
            }
        }
    }
    float s[PIX];
#pragma unroll
    for (int x = 0; x < PIX; ++x) {
        s[x] = 0.f;
#pragma unroll
        for (int c = 0; c < NC; ++c) s[x] = fmaf(acc[x][c].x, acc[x][c].x, fmaf(acc[x][c].y, acc[x][c].y, s[x]));
    }
    if constexpr (PIX == 2) reinterpret_cast<float2*>(a.M)[item] = make_float2(s[0], s[1]);
    else a.M[item] = s[0];
}

// complement (deflation) form; the T holograms of the thread's pixel(s) stay in registers and the
// rejected components are removed one after the other (modified Gram-Schmidt order):
//   for k not in S:  P = sum_t h_t V_tk ;  h_t -= P conj(V_tk)        then  M = sum_t |h_t|^2
template <int TMAX, int PIX>
__global__ void __launch_bounds__(256) k_project_deflate(const ProjArgs a, int nc) {
    extern __shared__ __align__(16) float2 Vd[];            // [c][TMAX], zero padded in t
    const int tid = threadIdx.x;
    const int n0 = a.r0_hi - a.r0_lo + 1 > 0 ? a.r0_hi - a.r0_lo + 1 : 0;
    for (int i = tid; i < nc * TMAX; i += blockDim.x) {
        const int c = i / TMAX, t = i - c * TMAX;
        const int col = c < n0 ? a.r0_lo + c : a.r1_lo + (c - n0);
        Vd[i] = t < a.T ? a.V[t * a.T + col] : make_float2(0.f, 0.f);
    }
    __syncthreads();
    const long long item = (long long)blockIdx.x * blockDim.x + tid;
    if (item * PIX >= a.npix) return;
    const long long fstride = a.npix / PIX;
    float2 h[TMAX][PIX];
#pragma unroll
    for (int t = 0; t < TMAX; ++t) {
        if (t < a.T) {
            if constexpr (PIX == 2) {
                const float4 w = __ldg(reinterpret_cast<const float4*>(a.H) + item + (long long)t * fstride);
                h[t][0] = make_float2(w.x, w.y); h[t][1] = make_float2(w.z, w.w);
            } else {
                h[t][0] = __ldg(a.H + item + (long long)t * fstride);
            }
        } else {
#pragma unroll
            for (int x = 0; x < PIX; ++x) h[t][x] = make_float2(0.f, 0.f);
        }
    }
    if (a.center) {
#pragma unroll
        for (int x = 0; x < PIX; ++x) {
            float2 m = make_float2(0.f, 0.f);
#pragma unroll
            for (int t = 0; t < TMAX; ++t) { m.x += h[t][x].x; m.y += h[t][x].y; }
            const float inv = 1.f / (float)a.T;
            m.x *= inv; m.y *= inv;
#pragma unroll
            for (int t = 0; t < TMAX; ++t) if (t < a.T) { h[t][x].x -= m.x; h[t][x].y -= m.y; }
        }
    }
#pragma unroll 1
    for (int c = 0; c < nc; ++c) {
        const float2* v = Vd + c * TMAX;
        float2 P[PIX];
#pragma unroll
        for (int x = 0; x < PIX; ++x) P[x] = make_float2(0.f, 0.f);
#pragma unroll
        for (int t = 0; t < TMAX; ++t) {
            const float2 w = v[t];
#pragma unroll
            for (int x = 0; x < PIX; ++x) {                       // P += h_t * v_t
                P[x].x = fmaf(h[t][x].x, w.x, fmaf(-h[t][x].y, w.y, P[x].x));
                P[x].y = fmaf(h[t][x].x, w.y, fmaf(h[t][x].y, w.x, P[x].y));
            }
        }
#pragma unroll
        for (int t = 0; t < TMAX; ++t) {
            const float2 w = v[t];
#pragma unroll
            for (int x = 0; x < PIX; ++x) {                       // h_t -= P * conj(v_t)
                h[t][x].x = fmaf(-P[x].x, w.x, fmaf(-P[x].y, w.y, h[t][x].x));
                h[t][x].y = fmaf(-P[x].y, w.x, fmaf(P[x].x, w.y, h[t][x].y));
            }
        }
    }
    float s[PIX];
#pragma unroll
    for (int x = 0; x < PIX; ++x) s[x] = 0.f;
#pragma unroll
    for (int t = 0; t < TMAX; ++t)
#pragma unroll
        for (int x = 0; x < PIX; ++x) s[x] = fmaf(h[t][x].x, h[t][x].x, fmaf(h[t][x].y, h[t][x].y, s[x]));
    if constexpr (PIX == 2) reinterpret_cast<float2*>(a.M)[item] = make_float2(s[0], s[1]);
    else a.M[item] = s[0];
}

// Deflation form fed by TMA: the same arithmetic as k_project_deflate, but the hologram stack is streamed
// into a shared-memory ring with 2-D tensor copies ([8 frames x 128 pixels] boxes, mbarrier complete_tx, one
// elected producer lane, 5-6 stages in flight) instead of T dependent 16-byte loads per thread.  Four
// consumer warps, one pixel per lane; a lane reads its pixel of every frame from shared memory (conflict
// free: 32 consecutive float2).  Bound by HBM; measured 4.7 -> see profiles/ TB/s.
// PROJ_P pixels per stage (256 up to T = 32, 128 above so that >= 2 stages fit); PROJ_P / 32 consumer warps
#define PROJ_MAX_STAGES 8
// HS = 2 (T > 32): TWO lanes per pixel, lanes l and l + 16 of a warp hold frames [0, TMAX/2) and [TMAX/2, TMAX) of pixel l & 15;
// the partial projections, means and energies are combined by one butterfly shuffle.  Twice the warps per stage (a single
// warp per scheduler at 255 registers was latency bound: 507 us at 2048^2 x 64) at half the registers.
template <int TMAX, int PROJ_P, int HS>
__global__ void __launch_bounds__(PROJ_P * HS, 1)
k_project_deflate_tma(const __grid_constant__ CUtensorMap tmH, const ProjArgs a, int nc, int nstages, int rb0, int nrb) {
    extern __shared__ __align__(128) unsigned char smraw[];
    uint64_t* full = reinterpret_cast<uint64_t*>(smraw);
    uint64_t* empty = full + PROJ_MAX_STAGES;
    float2* Vd = reinterpret_cast<float2*>(smraw + 128);                      // [nc][TMAX], zero padded in t
    const int vbytes = ((nc > 0 ? nc : 1) * TMAX * (int)sizeof(float2) + 127) & ~127;
    float2* ring = reinterpret_cast<float2*>(smraw + 128 + vbytes);           // [stage][TMAX][PROJ_P]
    constexpr int stage_elems = TMAX * PROJ_P;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const long long nchunks = a.npix / PROJ_P;
    const int n0 = a.r0_hi - a.r0_lo + 1 > 0 ? a.r0_hi - a.r0_lo + 1 : 0;
    for (int i = tid; i < nc * TMAX; i += blockDim.x) {
        const int c = i / TMAX, t = i - c * TMAX;
        const int col = c < n0 ? a.r0_lo + c : a.r1_lo + (c - n0);
        Vd[i] = t < a.T ? a.V[t * a.T + col] : make_float2(0.f, 0.f);
    }
    if (tid == 0) {
        for (int s = 0; s < nstages; ++s) { mbar_init(full + s, 1); mbar_init(empty + s, PROJ_P * HS / 32); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    // producer state (warp 0): rows >= T of the last box are zero-filled by the TMA unit
    int ps = 0; uint32_t pph = 0;
    long long pchunk = blockIdx.x;
    auto issue = [&]() {
        if (pchunk >= nchunks) return;
        mbar_wait(empty + ps, pph ^ 1u);
        if (lane == 0) mbar_arrive_expect_tx(full + ps, (uint32_t)stage_elems * (uint32_t)sizeof(float2));
        __syncwarp();
        // boxes of [8 frames x 128 pixels]; the stage is stored as PROJ_P/128 panels of [TMAX][128]
        if (lane < (TMAX / 8) * (PROJ_P / 128)) {
            const int rb = lane % (TMAX / 8), pan = lane / (TMAX / 8);
            tma_2d_g2s(ring + (size_t)ps * stage_elems + pan * (TMAX * 128) + rb * 8 * 128, &tmH,
                       (int)(pchunk * (2 * PROJ_P) + pan * 256), 8 * (nrb ? (rb0 + rb) % nrb : rb), full + ps);   // nrb != 0: ring window
        }
        pchunk += gridDim.x;
        if (++ps == nstages) { ps = 0; pph ^= 1u; }
    };
    if (warp == 0)
        for (int d = 0; d < nstages - 1; ++d) issue();
    int s = 0; uint32_t ph = 0;
    for (long long chunk = blockIdx.x; chunk < nchunks; chunk += gridDim.x) {
        mbar_wait(full + s, ph);
        constexpr int TH = TMAX / HS;                     // frames per thread
        // HS = 1: pixel = 32 warp + lane; HS = 2: pixel = 16 warp + (lane & 15), frames [TH (lane >> 4), + TH)
        const int pix = HS == 1 ? warp * 32 + lane : warp * 16 + (lane & 15);
        const int tb = HS == 1 ? 0 : (lane >> 4) * TH;
        const float2* src = ring + (size_t)s * stage_elems + (pix >> 7) * (TMAX * 128) + (pix & 127) + tb * 128;
        float2 h[TH];
#pragma unroll
        for (int t = 0; t < TH; ++t) h[t] = src[t * 128];
        __syncwarp();
        if (lane == 0) mbar_arrive(empty + s);           // the stage is in registers: hand it back at once
        if (warp == 0) issue();
        if (a.center) {                                   // rows t >= T are zero (TMA fill): they do not enter the mean
            float2 m = make_float2(0.f, 0.f);
#pragma unroll
            for (int t = 0; t < TH; ++t) { m.x += h[t].x; m.y += h[t].y; }
            if constexpr (HS == 2) { m.x += __shfl_xor_sync(0xffffffffu, m.x, 16); m.y += __shfl_xor_sync(0xffffffffu, m.y, 16); }
            const float inv = 1.f / (float)a.T;
            m.x *= inv; m.y *= inv;
#pragma unroll
            for (int t = 0; t < TH; ++t) if (tb + t < a.T) { h[t].x -= m.x; h[t].y -= m.y; }
        }
#pragma unroll 1
        for (int c = 0; c < nc; ++c) {
            const float2* v = Vd + c * TMAX + tb;
            float2 P = make_float2(0.f, 0.f);
#pragma unroll
            for (int t = 0; t < TH; ++t) {                        // P += h_t * v_t
                const float2 w = v[t];
                P.x = fmaf(h[t].x, w.x, fmaf(-h[t].y, w.y, P.x));
                P.y = fmaf(h[t].x, w.y, fmaf(h[t].y, w.x, P.y));
            }
            if constexpr (HS == 2) { P.x += __shfl_xor_sync(0xffffffffu, P.x, 16); P.y += __shfl_xor_sync(0xffffffffu, P.y, 16); }
#pragma unroll
            for (int t = 0; t < TH; ++t) {                        // h_t -= P * conj(v_t)
                const float2 w = v[t];
                h[t].x = fmaf(-P.x, w.x, fmaf(-P.y, w.y, h[t].x));
                h[t].y = fmaf(-P.y, w.x, fmaf(P.x, w.y, h[t].y));
            }
        }
        float sum = 0.f;
#pragma unroll
        for (int t = 0; t < TH; ++t) sum = fmaf(h[t].x, h[t].x, fmaf(h[t].y, h[t].y, sum));
        if constexpr (HS == 2) sum += __shfl_xor_sync(0xffffffffu, sum, 16);
        if (HS == 1 || lane < 16) a.M[chunk * PROJ_P + pix] = sum;
        if (++s == nstages) { s = 0; ph ^= 1u; }
    }
}

template <int TMAX> static int launch_deflate(holo_ctx* c, const ProjArgs& a, int nc, cudaStream_t st) {
    constexpr int PROJ_P = TMAX <= 32 ? 256 : 128;
    constexpr int HS = TMAX <= 32 ? 1 : 2;             // lanes per pixel (T > 32: the frames of a pixel are split over two lanes)
    const int vbytes = ((nc > 0 ? nc : 1) * TMAX * (int)sizeof(float2) + 127) & ~127;
    const size_t stage_bytes = (size_t)TMAX * PROJ_P * sizeof(float2);
    int nstages = (int)((200 * 1024 - vbytes) / stage_bytes);
    if (nstages > PROJ_MAX_STAGES) nstages = PROJ_MAX_STAGES;
    if (c->ring_nrb && !(c->tune[HOLO_TUNE_PROJ_TMA] && nstages >= 2 && a.npix % PROJ_P == 0 && a.T == TMAX)) {
        holo_set_error("ring projection needs the TMA kernel and T in {8,16,32,64}"); return HOLO_ERR_STATE;
    }
    if (c->tune[HOLO_TUNE_PROJ_TMA] && nstages >= 2 && a.npix % PROJ_P == 0) {
        const size_t smem = 128 + vbytes + (size_t)nstages * stage_bytes;
        { const int rc = holo_ensure_smem_attr((const void*)k_project_deflate_tma<TMAX, PROJ_P, HS>, c->device, 200 * 1024 + 128); if (rc) return rc; }
        alignas(64) CUtensorMap tmH;
        { const int rc = holo_make_tensor_map(&tmH, a.H, a.npix, c->ring_nrb ? 8 * c->ring_nrb : a.T, 128); if (rc) return rc; }
        const long long nchunks = a.npix / PROJ_P;
        const int cap = c->proj_grid_cap > 0 ? c->proj_grid_cap : c->num_sms;
        const int grid = (int)(nchunks < cap ? nchunks : cap);
        HoloProf prof(c, HOLO_K_PROJECT, st);
        k_project_deflate_tma<TMAX, PROJ_P, HS><<<grid, PROJ_P * HS, smem, st>>>(tmH, a, nc, nstages, c->ring_rb0, c->ring_nrb);
        HOLO_CUDA_OK(cudaGetLastError());
        return HOLO_OK;
    }
    HoloProf prof(c, HOLO_K_PROJECT, st);
    constexpr int PIX = TMAX <= 32 ? 2 : 1;
    const long long items = a.npix / PIX;
    const int threads = 256;
    const int grid = (int)((items + threads - 1) / threads);
    const size_t smem = (size_t)(nc > 0 ? nc : 1) * TMAX * sizeof(float2);
    k_project_deflate<TMAX, PIX><<<grid, threads, smem, st>>>(a, nc);
    HOLO_CUDA_OK(cudaGetLastError());
    return HOLO_OK;
}

template <int NC> static int launch_proj_t(holo_ctx* c, const ProjArgs& a, cudaStream_t st) {
    HoloProf prof(c, HOLO_K_PROJECT, st);
    constexpr int PIX = NC > 32 ? 1 : 2;
    const long long items = a.npix / PIX;
    const int threads = 256;
    const int grid = (int)((items + threads - 1) / threads);
    k_project<NC, PIX><<<grid, threads, 0, st>>>(a);
    HOLO_CUDA_OK(cudaGetLastError());
    return HOLO_OK;
}

int holo_launch_project(holo_ctx* c, const float2* H, const float2* V, int k_lo, int k_hi,
                        int allow_complement, float* image, cudaStream_t st, int center) {
    const int T = c->T;
    const int nS = k_hi - k_lo + 1;
    ProjArgs a{};
    a.H = H; a.V = V; a.M = image; a.npix = c->npix; a.T = T; a.center = center;
    int nc;
    if (allow_complement && 2 * (T - nS) <= nS) {          // deflating costs 2 passes per rejected component
        a.complement = 1;
        a.r0_lo = 0; a.r0_hi = k_lo - 2;          // components 1 .. k_lo-1
        a.r1_lo = k_hi; a.r1_hi = T - 1;          // components k_hi+1 .. T
        nc = T - nS;
    } else {
        a.complement = 0;
        a.r0_lo = k_lo - 1; a.r0_hi = k_hi - 1;
        a.r1_lo = 0; a.r1_hi = -1;
        nc = nS;
    }
    if (center && !a.complement) { holo_set_error("the centred projection needs the deflation form (rejected set at most half of the kept set)"); return HOLO_ERR_STATE; }
    if (a.complement) {
        if (T <= 8) return launch_deflate<8>(c, a, nc, st);
        if (T <= 16) return launch_deflate<16>(c, a, nc, st);
        if (T <= 32) return launch_deflate<32>(c, a, nc, st);
        return launch_deflate<64>(c, a, nc, st);
    }
    if (nc > 4 && !c->ring_nrb && c->tune[HOLO_TUNE_PROJ_TC] && holo_project_tc_supported(c, nc))
        return holo_launch_project_tc(c, H, V, k_lo, k_hi, image, st);
    if (nc <= 1) return launch_proj_t<1>(c, a, st);
    if (nc <= 2) return launch_proj_t<2>(c, a, st);
    if (nc <= 4) return launch_proj_t<4>(c, a, st);
    if (nc <= 8) return launch_proj_t<8>(c, a, st);
    if (nc <= 16) return launch_proj_t<16>(c, a, st);
    if (nc <= 32) return launch_proj_t<32>(c, a, st);
    return launch_proj_t<64>(c, a, st);
}
