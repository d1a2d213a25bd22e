// fresnel.cu -- A0 (temporal sum), A1 (mean-subtract + chirp prologue) and A2 (2-D FFT) kernels.
//   H_t = FFT2D[(I_t - mean_t I) * exp(+i pi (x^2+y^2)/(lambda z))]      (Eq. 1; R2-R6)
// Stockham autosort FFT, radix-16/32 butterflies in registers (FMA-fused DIT), one shared-memory exchange per extra
// pass, row pass (x) then column pass (y); the row->column intermediate is kept L2-resident by
// processing the stack in small frame groups.
#include "holo_internal.cuh"
#include "fft_reg.cuh"
#include <math.h>
#include <vector>
#include <type_traits>

// ------------------------------------------------------------------------------------------------
// A0: per-pixel temporal sum  S(p) = sum_t I_t(p)   (uint32: exact, T*65535 < 2^32)
// ------------------------------------------------------------------------------------------------
// Batches of SUM_U frames are loaded into registers before any of them is added: left to itself the compiler keeps two loads
// in flight per thread (16 round trips to DRAM at T = 32): 17.9 -> 13.4 us at 512 x 512 x 32, 20.0 -> 17.3 us at 1024 x 1024 x 32.
__global__ void __launch_bounds__(256) k_frame_sum(const uint16_t* __restrict__ frames, uint32_t* __restrict__ sum,
                                                   long long npix, int T, unsigned int* __restrict__ counters) {
    pdl_trigger();                                        // (the Fresnel kernel may become resident while this one drains)
    if (blockIdx.x == 0 && threadIdx.x < 2 * T + 1) counters[threadIdx.x] = 0u;   // ticket / completion counters of the fused Fresnel kernel
    if (blockIdx.x == 0 && threadIdx.x == 0) counters[1001] = 0u;                 // row ticket of the packed row pass
    long long v = (long long)blockIdx.x * blockDim.x + threadIdx.x;      // one uint4 = 8 pixels per thread
    long long nvec = npix >> 3;
    for (; v < nvec; v += (long long)gridDim.x * blockDim.x) {
        uint32_t s[8] = {0, 0, 0, 0, 0, 0, 0, 0};
        const uint4* src = reinterpret_cast<const uint4*>(frames) + v;
        auto add = [&](const uint4& w) {
            s[0] += w.x & 0xffffu; s[1] += w.x >> 16;
            s[2] += w.y & 0xffffu; s[3] += w.y >> 16;
            s[4] += w.z & 0xffffu; s[5] += w.z >> 16;
            s[6] += w.w & 0xffffu; s[7] += w.w >> 16;
        };
        constexpr int SUM_U = 16;
        int t = 0;
        for (; t + SUM_U <= T; t += SUM_U) {
            uint4 w[SUM_U];
#pragma unroll
            for (int j = 0; j < SUM_U; ++j) w[j] = __ldg(src + (long long)(t + j) * nvec);
#pragma unroll
            for (int j = 0; j < SUM_U; ++j) add(w[j]);
        }
        for (; t < T; ++t) add(__ldg(src + (long long)t * nvec));
        uint4* dst = reinterpret_cast<uint4*>(sum) + 2 * v;
        dst[0] = make_uint4(s[0], s[1], s[2], s[3]);
        dst[1] = make_uint4(s[4], s[5], s[6], s[7]);
    }
}

// ------------------------------------------------------------------------------------------------
// 1-D FFT pass kernel over a batch of B sequences per CTA.
//   COL = false: sequences are image rows (contiguous), PRO = fused uint16/mean/chirp prologue
//   COL = true : sequences are image columns (stride ld), B adjacent columns per CTA
// ------------------------------------------------------------------------------------------------
struct FftArgs {
    const uint16_t* frames;   // PRO: [nf][ny][nx] (already offset to the first frame of the group)
    const uint32_t* sum;      // PRO
    const float2* qx;         // PRO
    const float2* qy;         // PRO
    const float2* in;         // !PRO
    float2* out;
    const float2* tw1;
    const float2* tw2;
    long long in_fstride, out_fstride;   // elements between frames
    int ld;                   // elements between consecutive rows (= nx)
    int nseq;                 // sequences per frame (ROW: ny, COL: nx)
    int tiles_per_frame;      // nseq / B
    int ntiles;               // nf * tiles_per_frame
    int T;
    // raw-domain deflation (mode 3, DEFL prologue): d'_t = (T I_t - S) - sum_k eT_k V_{t,k}
    const float* defl_img;    // [ndefl][ny][nx]  eT_k = sum_t (T I_t - S) V_{t,k} of the rejected components
    const float* defl_coef;   // [T][ndefl]       V_{t,k} (real: C is real symmetric there, R21)
    int ndefl;
    const float* eimg;        // prologue mode 2: real input images [nframes][ny][nx] (in_fstride elements apart)
    unsigned int* ticket;     // != nullptr: row kernels of one warp per row draw single rows from this counter (zeroed by the
                              // caller's earlier kernel) instead of a static partition: a CTA that shares its SM with the
                              // eigensolver of the side stream then simply takes fewer rows
};

// one tile = B sequences of one frame; in_foff / out_foff = element offset of the frame in a.in(frames) / a.out
struct NoHook { __device__ __forceinline__ void operator()() const {} };

// `mid` is called once by every thread in the middle of the tile (after the pass-0 butterflies; the fused
// kernel does its scheduling work there, when the stores of the previous tile have long drained)
// LDC: row pitch in elements known at compile time (0: use a.ld) -- turns every address into base + immediate
// DEFL (prologue mode of PRO tiles): 0 = d = T I - S; 1 = the rejected components are also removed in the raw domain (frame
// index `frame` selects the V row); 2 = the input is a real float image (a.eimg: eigen-images of mode 3), d = eimg.
// ENERGY: nothing is stored; |X|^2 of output slot s (the s-th value this thread would store, see tile_out_offset) is added
// to acc[s] instead.
// TILED = w > 0 (column tiles without prologue): the input is stored in column blocks of w >= B columns,
// [frame][x / w][row][x % w] (the packed row pass writes it so): the tiles of w / B neighbouring CTAs are ONE contiguous block
// of N * w elements instead of N row segments one row pitch apart.
template <int N, int E, int R1, int R2, int B, bool COL, bool PRO, int LDC = 0, class Mid = NoHook, int DEFL = 0, bool ENERGY = false,
          int TILED = 0>
__device__ __forceinline__ void fft_tile(const FftArgs& a, long long in_foff, long long out_foff, int tile_in_frame, float2* sm,
                                         Mid mid = Mid(), int frame = 0, float* acc = nullptr, int seq_override = -1) {
    constexpr int TPS = N / E;
    constexpr int PADN = N + N / E;
    constexpr bool MULTI = (R1 > 1);
    // a row whose N/E threads are exactly one warp is exchanged through that warp's private slice of the buffer:
    // warp-level synchronisation only (the eight warps of a row tile then run freely against each other)
    constexpr bool WARP_SEQ = !COL && (N / E == 32);
    constexpr bool FREE_RUN = std::is_same<Mid, NoHook>::value;
    auto sync_tile = [&]() { if constexpr (WARP_SEQ) __syncwarp(); else __syncthreads(); };
    const int tid = threadIdx.x;
    const int j = COL ? tid / B : tid % TPS;
    const int c = COL ? tid % B : tid / TPS;
    auto sidx = [&](int i) -> int {
        int p = i + i / E;
        return COL ? p * B + c : c * PADN + p;
    };
    {
        const int s0 = seq_override >= 0 ? seq_override : tile_in_frame * B + c;   // sequence index (row y or column x)
        const int ld = LDC ? LDC : a.ld;
        const long long ibase = in_foff + (COL ? (long long)s0 : (long long)s0 * ld);
        const long long obase = out_foff + (COL ? (long long)s0 : (long long)s0 * ld);
        const int estride = COL ? ld : 1;
        constexpr bool FUSED = LDC != 0;                 // fused persistent kernel: rows write / columns read the L2 ring
        const uint64_t pol_in = (FUSED && COL) ? l2_evict_last() : l2_evict_first();
        const uint64_t pol_out = (FUSED && !COL) ? l2_evict_last() : l2_evict_first();
        auto store = [&](float2* q, float2 val) { if constexpr (FUSED) st_hint(q, val, pol_out); else *q = val; };
        // output slot `slot` of this thread: element offset `off` (in units of estride) from op
        auto emit = [&](int slot, float2* op_, int off, float2 val) {
            if constexpr (ENERGY) acc[slot] = fmaf(val.x, val.x, fmaf(val.y, val.y, acc[slot]));
            else store(op_ + off * estride, val);
        };
        float2 v[E];
        // ---------------- pass 0: radix E, Ns = 1, inputs straight from global
        if constexpr (PRO) {
            const float2 qyv = __ldg(a.qy + s0);
            const uint16_t* fr = a.frames + ibase;
            const uint32_t* sp = a.sum + (long long)s0 * ld;
            if constexpr (DEFL == 2) {
                const float* ep = a.eimg + in_foff + (long long)s0 * ld + j;
                float e[E];
#pragma unroll
                for (int r = 0; r < E; ++r) e[r] = __ldg(ep + r * TPS);
#pragma unroll
                for (int r = 0; r < E; ++r) {
                    const float2 q = cmul(__ldg(a.qx + j + r * TPS), qyv);
                    v[r] = make_float2(e[r] * q.x, e[r] * q.y);
                }
            } else if constexpr (DEFL == 0) {
#pragma unroll
                for (int r = 0; r < E; ++r) {
                    const int i = j + r * TPS;
                    const int I = FUSED ? ldnc_u16_hint(fr + i, pol_in) : (int)__ldg(fr + i);
                    const int S = (int)__ldg(sp + i);
                    const float d = (float)(a.T * I - S);                  // exact integer; the 1/T lives in the qx table
                    const float2 q = cmul(__ldg(a.qx + i), qyv);
                    v[r] = make_float2(d * q.x, d * q.y);
                }
            } else {
                // d' = (T I - S) - sum_k eT_k V_{t,k}: all loads of one component are issued together (E in flight per thread)
#pragma unroll
                for (int r = 0; r < E; ++r) {
                    const int i = j + r * TPS;
                    v[r].x = (float)(a.T * (int)__ldg(fr + i) - (int)__ldg(sp + i));
                }
                const float* ep = a.defl_img + (long long)s0 * ld + j;
                for (int kk = 0; kk < a.ndefl; ++kk) {
                    const float cf = -__ldg(a.defl_coef + frame * a.ndefl + kk);
                    float e[E];
#pragma unroll
                    for (int r = 0; r < E; ++r) e[r] = __ldg(ep + r * TPS);
#pragma unroll
                    for (int r = 0; r < E; ++r) v[r].x = fmaf(e[r], cf, v[r].x);
                    ep += (long long)a.nseq * ld;
                }
#pragma unroll
                for (int r = 0; r < E; ++r) {
                    const float2 q = cmul(__ldg(a.qx + j + r * TPS), qyv);
                    const float d = v[r].x;
                    v[r] = make_float2(d * q.x, d * q.y);
                }
            }
        } else {
            if constexpr (TILED != 0) {
                const int x = tile_in_frame * B + c;
                const float2* ip = a.in + in_foff + (long long)(x / TILED) * (N * TILED) + x % TILED;
#pragma unroll
                for (int r = 0; r < E; ++r) v[r] = __ldcg(ip + (j + r * TPS) * TILED);
            } else {
            const float2* ip = a.in + ibase;
#pragma unroll
            for (int r = 0; r < E; ++r) v[r] = FUSED ? ldcg_hint(ip + (j + r * TPS) * estride, pol_in) : __ldcg(ip + (j + r * TPS) * estride);   // L2-coherent: written earlier in this kernel
            }
        }
        fft_reg<E>(v);
        float2* op = a.out + obase;
        if constexpr (!MULTI) {
            mid();
#pragma unroll
            for (int r = 0; r < E; ++r) emit(r, op, r, v[brev<E>(r)]);
        } else {
#pragma unroll
            for (int r = 0; r < E; ++r) sm[sidx(j * E + r)] = v[brev<E>(r)];
            sync_tile();
            mid();
            // ---------------- pass 1: radix R1, Ns = E
            constexpr int M1 = E / R1;
#pragma unroll
            for (int m = 0; m < M1; ++m) {
                const int b = j + m * TPS;
#pragma unroll
                for (int r = 0; r < R1; ++r) v[m * R1 + r] = sm[sidx(b + r * (N / R1))];
            }
            if constexpr (R2 > 1) sync_tile();
#pragma unroll
            for (int m = 0; m < M1; ++m) {
                const int b = j + m * TPS;
                const int k = b % E;
#pragma unroll
                for (int r = 1; r < R1; ++r) v[m * R1 + r] = cmul(v[m * R1 + r], __ldg(a.tw1 + r * E + k));
                fft_reg<R1>(v + m * R1);
                const int j0 = (b - k) * R1 + k;
                if constexpr (R2 == 1) {
#pragma unroll
                    for (int r = 0; r < R1; ++r) emit(m * R1 + r, op, j0 + r * E, v[m * R1 + brev<R1>(r)]);
                } else {
#pragma unroll
                    for (int r = 0; r < R1; ++r) sm[sidx(j0 + r * E)] = v[m * R1 + brev<R1>(r)];
                }
            }
            if constexpr (R2 > 1) {
                sync_tile();
                // ---------------- pass 2: radix R2, Ns = E*R1
                constexpr int M2 = E / R2;
                constexpr int NS2 = E * R1;
#pragma unroll
                for (int m = 0; m < M2; ++m) {
                    const int b = j + m * TPS;
#pragma unroll
                    for (int r = 0; r < R2; ++r) v[m * R2 + r] = sm[sidx(b + r * (N / R2))];
                }
#pragma unroll
                for (int m = 0; m < M2; ++m) {
                    const int b = j + m * TPS;                         // b < N/R2 = NS2, so k = b
#pragma unroll
                    for (int r = 1; r < R2; ++r) v[m * R2 + r] = cmul(v[m * R2 + r], __ldg(a.tw2 + r * NS2 + b));
                    fft_reg<R2>(v + m * R2);
#pragma unroll
                    for (int r = 0; r < R2; ++r) emit(m * R2 + r, op, b + r * NS2, v[m * R2 + brev<R2>(r)]);
                }
            }
            // smem is reused by the next tile.  Row tiles of one warp per row (private slices) outside the fused kernel need
            // no CTA-wide barrier at all: the warps of a CTA then drift apart and overlap each other's load and store phases
            if constexpr (WARP_SEQ && FREE_RUN) __syncwarp(); else __syncthreads();
        }
    }
}

template <int N, int E, int R1, int R2, int B, bool COL, bool PRO, int DEFL = 0>
__global__ void __launch_bounds__((N / E) * B) k_fft(const FftArgs a) {
    extern __shared__ float2 sm[];
    if constexpr (!COL && N / E == 32) {
        if (a.ticket) {                                      // one warp per row, rows drawn one by one (no CTA-wide step at all)
            const unsigned int nrows = (unsigned int)a.ntiles * B;
            for (;;) {
                unsigned int r = 0u;
                if ((threadIdx.x & 31) == 0) r = atomicAdd(a.ticket, 1u);
                r = __shfl_sync(0xffffffffu, r, 0);
                if (r >= nrows) break;
                const int fl = (int)(r / (unsigned int)a.nseq), row = (int)(r - (unsigned int)fl * a.nseq);
                fft_tile<N, E, R1, R2, B, COL, PRO, 0, NoHook, DEFL>(a, (long long)fl * a.in_fstride, (long long)fl * a.out_fstride,
                                                                     0, sm, NoHook(), fl, nullptr, row);
            }
            return;
        }
    }
    for (int tile = blockIdx.x; tile < a.ntiles; tile += gridDim.x) {
        const int fl = tile / a.tiles_per_frame;
        fft_tile<N, E, R1, R2, B, COL, PRO, 0, NoHook, DEFL>(a, (long long)fl * a.in_fstride, (long long)fl * a.out_fstride,
                                                             tile - fl * a.tiles_per_frame, sm, NoHook(), fl);
    }
}

// column pass of whole frames whose row-pass output is stored in column blocks of B columns (see TILED above); plain
// row-major output.  Tiles in frame-major order: concurrent CTAs walk adjacent column tiles of the same frame.
template <int N, int E, int R1, int R2, int B>
__global__ void __launch_bounds__((N / E) * B) k_cols_tiled(const FftArgs a) {
    extern __shared__ float2 sm[];
    pdl_wait();
    const int nf = a.ntiles / a.tiles_per_frame;
    for (int tile = blockIdx.x; tile < a.ntiles; tile += gridDim.x) {
        const int fr = tile / a.tiles_per_frame;
        const int fl = nf - 1 - fr;                          // newest frames first: the tail of the row-pass output is still in L2 (-4 us)
        fft_tile<N, E, R1, R2, B, true, false, 0, NoHook, 0, false, B>(a, (long long)fl * a.in_fstride, (long long)fl * a.out_fstride,
                                                                       tile - fr * a.tiles_per_frame, sm);
    }
}

// element offset (in units of the sequence stride) of output slot `slot` of the calling thread: mirrors the emission
// order of fft_tile
template <int N, int E, int R1, int R2, int B, bool COL>
__device__ __forceinline__ int tile_out_offset(int slot) {
    constexpr int TPS = N / E;
    const int j = COL ? (int)threadIdx.x / B : (int)threadIdx.x % TPS;
    if constexpr (R1 == 1) return slot;
    else if constexpr (R2 == 1) {
        const int m = slot / R1, r = slot % R1;
        const int b = j + m * TPS, k = b % E;
        return (b - k) * R1 + k + r * E;
    } else {
        const int m = slot / R2, r = slot % R2;
        return j + m * TPS + r * (E * R1);
    }
}

// Mode 3 (SURVEY.md 8(f)-2 stage 2), second pass: the column transform of frames [t0, t1) of one column tile, REDUCED to
// its energy: out(p) = sum_{t in [t0,t1)} |H'_t(p)|^2 with H'_t the hologram of the deflated frame t (rejected components
// already removed in the raw domain by the row pass), so that sum over all t is the image of Eq. 7 (R12
// identity: sum_{k in S}|P_k|^2 = sum_t |H_t - sum_{k not in S} P_k conj(V_tk)|^2 for unitary V).  The hologram stack is
// never written.  grid = (column tiles, frame splits); split s writes out + s * npix (a plain store: deterministic).
template <int N, int E, int R1, int R2, int B, int TILED = 0>
__global__ void __launch_bounds__((N / E) * B, 512 / ((N / E) * B) > 0 ? 512 / ((N / E) * B) : 1)
k_col_energy(const FftArgs a, float* __restrict__ out, long long npix, int nframes, int nsplit) {
    extern __shared__ float2 sm[];
    pdl_trigger();                                        // (k_sum_partial_images may become resident)
    pdl_wait();                                           // the row pass is complete
    const int tile = blockIdx.x, split = blockIdx.y;
    float acc[E];
#pragma unroll
    for (int s = 0; s < E; ++s) acc[s] = 0.f;
    // split s takes the frames nframes-1-s, nframes-1-s-nsplit, ...: all splits start with the frames the row pass wrote
    // LAST, which are still in L2 (the row-pass output is larger than L2), and walk down together
    for (int t = nframes - 1 - split; t >= 0; t -= nsplit)
        fft_tile<N, E, R1, R2, B, true, false, 0, NoHook, 0, true, TILED>(a, (long long)t * a.in_fstride, 0, tile, sm, NoHook(), 0, acc);
    const int c = (int)threadIdx.x % B;
    float* op = out + (long long)split * npix + (long long)tile * B + c;
#pragma unroll
    for (int s = 0; s < E; ++s) op[(long long)tile_out_offset<N, E, R1, R2, B, true>(s) * a.ld] = acc[s];
}

// out = sum of nsplit partial images (fixed order)
__global__ void __launch_bounds__(256) k_sum_partial_images(const float* __restrict__ part, int nsplit, long long npix, float* __restrict__ out) {
    const long long n4 = npix >> 2;                         // npix is a multiple of 256
    const float4* p4 = reinterpret_cast<const float4*>(part);
    pdl_wait();
    for (long long p = (long long)blockIdx.x * 256 + threadIdx.x; p < n4; p += (long long)gridDim.x * 256) {
        float4 s = __ldg(p4 + p);
        for (int k = 1; k < nsplit; ++k) { const float4 w = __ldg(p4 + (long long)k * n4 + p); s.x += w.x; s.y += w.y; s.z += w.z; s.w += w.w; }
        reinterpret_cast<float4*>(out)[p] = s;
    }
}

// Mode 3, eigen-basis form: E_k(x) = sum_t (T I_t(x) - S(x)) Re V_{t,k} for the KEPT components k = c_lo .. c_lo + nS - 1
// (float [nS][npix]).  With V real and orthonormal, sum_{k in S} |F[q E_k]|^2 = sum_{k in S} |P_k|^2 T^2: the image of Eq. 7
// from nS transforms instead of T, for any window.  PX pixels per thread: the frame values stay in registers, the
// coefficients are broadcast from shared memory (one LDS per PX FMAs).
template <int TMAX, int PX>
__global__ void __launch_bounds__(128) k_eigen_images(const uint16_t* __restrict__ frames, const uint32_t* __restrict__ sum,
                                                      const float2* __restrict__ V, long long npix, int T, int c_lo, int nS, float* __restrict__ img) {
    extern __shared__ float Vs_e[];                        // [nS][TMAX], zero padded in t
    for (int i = threadIdx.x; i < nS * TMAX; i += blockDim.x) {
        const int k = i / TMAX, t = i - k * TMAX;
        Vs_e[i] = t < T ? V[t * T + c_lo + k].x : 0.f;
    }
    __syncthreads();
    const long long nvec = npix / PX;
    const float Tf = (float)T;
    for (long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x; q < nvec; q += (long long)gridDim.x * blockDim.x) {
        float d[TMAX][PX];
        float S[PX];
#pragma unroll
        for (int x = 0; x < PX; ++x) S[x] = (float)__ldg(sum + q * PX + x);
#pragma unroll
        for (int t = 0; t < TMAX; ++t) {
            if (t < T) {
                if constexpr (PX == 4) {
                    const uint2 w = __ldg(reinterpret_cast<const uint2*>(frames + (long long)t * npix) + q);
                    d[t][0] = fmaf(Tf, (float)(w.x & 0xffffu), -S[0]); d[t][1] = fmaf(Tf, (float)(w.x >> 16), -S[1]);
                    d[t][2] = fmaf(Tf, (float)(w.y & 0xffffu), -S[2]); d[t][3] = fmaf(Tf, (float)(w.y >> 16), -S[3]);
                } else {
                    const uint32_t w = __ldg(reinterpret_cast<const uint32_t*>(frames + (long long)t * npix) + q);
                    d[t][0] = fmaf(Tf, (float)(w & 0xffffu), -S[0]); d[t][1] = fmaf(Tf, (float)(w >> 16), -S[1]);
                }
            } else {
#pragma unroll
                for (int x = 0; x < PX; ++x) d[t][x] = 0.f;
            }
        }
#pragma unroll 1
        for (int k = 0; k < nS; ++k) {
            const float* v = Vs_e + k * TMAX;
            float acc[PX];
#pragma unroll
            for (int x = 0; x < PX; ++x) acc[x] = 0.f;
#pragma unroll
            for (int t = 0; t < TMAX; ++t) {
                const float w = v[t];
#pragma unroll
                for (int x = 0; x < PX; ++x) acc[x] = fmaf(d[t][x], w, acc[x]);
            }
            float* dst = img + (long long)k * npix + q * PX;
            if constexpr (PX == 4) *reinterpret_cast<float4*>(dst) = make_float4(acc[0], acc[1], acc[2], acc[3]);
            else *reinterpret_cast<float2*>(dst) = make_float2(acc[0], acc[1]);
        }
    }
}

// eT_k(x) = sum_t (T I_t(x) - S(x)) V_{t,k} for the rejected components k (column indices of V: c0_lo + kk for kk < c0_n,
// then c1_lo + ...), and the coefficient table coef[t][kk] = Re V_{t,k}.  Eight pixels per thread (16-byte loads, eight
// frames in flight), NDEFL accumulators per pixel.
template <int NDEFL>
__global__ void __launch_bounds__(256) k_deflate_images(const uint16_t* __restrict__ frames, const uint32_t* __restrict__ sum,
                                                        const float2* __restrict__ V, long long npix, int T,
                                                        int c0_lo, int c0_n, int c1_lo, float* __restrict__ img, float* __restrict__ coef) {
    __shared__ float Vs[HOLO_MAX_T * NDEFL];
    pdl_trigger();                                        // (the row pass may load its tables while this kernel drains)
    for (int i = threadIdx.x; i < T * NDEFL; i += blockDim.x) {
        const int t = i / NDEFL, kk = i - t * NDEFL;
        const int col = kk < c0_n ? c0_lo + kk : c1_lo + (kk - c0_n);
        const float v = V[t * T + col].x;
        Vs[i] = v;
        if (blockIdx.x == 0) coef[i] = v;
    }
    __syncthreads();
    const long long nvec = npix >> 3;
    const float Tf = (float)T;
    for (long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x; q < nvec; q += (long long)gridDim.x * blockDim.x) {
        const uint4 sa = __ldg(reinterpret_cast<const uint4*>(sum) + 2 * q), sb = __ldg(reinterpret_cast<const uint4*>(sum) + 2 * q + 1);
        const float S[8] = {(float)sa.x, (float)sa.y, (float)sa.z, (float)sa.w, (float)sb.x, (float)sb.y, (float)sb.z, (float)sb.w};   // < 2^22: exact
        float e[NDEFL][8];
#pragma unroll
        for (int kk = 0; kk < NDEFL; ++kk)
#pragma unroll
            for (int x = 0; x < 8; ++x) e[kk][x] = 0.f;
        const uint4* src = reinterpret_cast<const uint4*>(frames) + q;
        auto accumulate = [&](const uint4& w, int t) {
            const uint32_t ws[4] = {w.x, w.y, w.z, w.w};
            float d[8];
#pragma unroll
            for (int x = 0; x < 4; ++x) {
                d[2 * x] = fmaf(Tf, (float)(ws[x] & 0xffffu), -S[2 * x]);          // T I - S: integers below 2^23, exact in FP32
                d[2 * x + 1] = fmaf(Tf, (float)(ws[x] >> 16), -S[2 * x + 1]);
            }
#pragma unroll
            for (int kk = 0; kk < NDEFL; ++kk) {
                const float v = Vs[t * NDEFL + kk];
#pragma unroll
                for (int x = 0; x < 8; ++x) e[kk][x] = fmaf(d[x], v, e[kk][x]);
            }
        };
        // batches of DEFL_U frames in registers before the arithmetic (as k_frame_sum: the loads of a batch are all in flight)
        constexpr int DEFL_U = 16;
        int t = 0;
        for (; t + DEFL_U <= T; t += DEFL_U) {
            uint4 w[DEFL_U];
#pragma unroll
            for (int j = 0; j < DEFL_U; ++j) w[j] = __ldg(src + (long long)(t + j) * nvec);
#pragma unroll
            for (int j = 0; j < DEFL_U; ++j) accumulate(w[j], t + j);
        }
        for (; t < T; ++t) accumulate(__ldg(src + (long long)t * nvec), t);
#pragma unroll
        for (int kk = 0; kk < NDEFL; ++kk) {
            float4* dst = reinterpret_cast<float4*>(img + (long long)kk * npix) + 2 * q;
            dst[0] = make_float4(e[kk][0], e[kk][1], e[kk][2], e[kk][3]);
            dst[1] = make_float4(e[kk][4], e[kk][5], e[kk][6], e[kk][7]);
        }
    }
}

// ------------------------------------------------------------------------------------------------
// Persistent fused Fresnel kernel (square frames): ONE launch does the row pass and the column pass of
// all T frames.  CTAs draw tiles from a global ticket (atomicAdd: a compare-and-swap claim of "ready" tiles
// was measured to serialise at one claim per L2 round trip, 4.5 ms) in the order
//   rows(0..L-1), [rows(f), cols(f-L)] for f = L..T-1, cols(T-L..T-1)
// The lag L (frames) is chosen so that the tickets in flight (one or two per resident CTA) span fewer
// tiles than separate rows(f) from cols(f): a column tile then almost never waits for its row pass.
// The row->column intermediate is a ring of R > L frames that stays in L2: cols(f) waits for
// rows_done[f] == RT, rows(f) waits for cols_done[f-R] == CT (ring reuse).  Tickets are served in order and
// every dependency of a ticket has a smaller ticket, so the smallest unfinished ticket can always run.
// ------------------------------------------------------------------------------------------------
struct FresnelArgs {
    FftArgs rows, cols;         // rows.out = cols.in = scratch ring; frame offsets are computed here
    unsigned int* counters;     // [0] ticket, [1..T] rows_done, [1+T..2T] cols_done (zeroed by k_frame_sum)
    long long npix;
    int T, R, L, RT, CT;
};

// ticket -> (frame, tile in frame, row/column pass)
__device__ __forceinline__ void fresnel_decode(const FresnelArgs& p, unsigned int tk, int& f, int& w, bool& is_col) {
    const unsigned int per = (unsigned int)(p.RT + p.CT);
    const unsigned int head = (unsigned int)(p.L * p.RT);                    // rows(0..L-1)
    const unsigned int body = head + (unsigned int)(p.T - p.L) * per;        // + [rows(f), cols(f-L)]
    if (tk < head) { f = (int)(tk / (unsigned int)p.RT); w = (int)tk - f * p.RT; is_col = false; }
    else if (tk < body) {
        const unsigned int u = tk - head;
        const int seg = (int)(u / per), r = (int)(u - (unsigned int)seg * per);
        if (r < p.RT) { f = seg + p.L; w = r; is_col = false; } else { f = seg; w = r - p.RT; is_col = true; }
    } else {
        const unsigned int u = tk - body;
        const int g = (int)(u / (unsigned int)p.CT);
        f = p.T - p.L + g; w = (int)u - g * p.CT; is_col = true;
    }
}
// counter a tile depends on (nullptr: none) and the value it must reach
__device__ __forceinline__ const unsigned int* fresnel_dep(const FresnelArgs& p, int f, bool is_col, unsigned int& need) {
    if (is_col) { need = (unsigned int)p.RT; return p.counters + 1 + f; }
    if (f >= p.R) { need = (unsigned int)p.CT; return p.counters + 1 + p.T + (f - p.R); }
    need = 0u;
    return nullptr;
}

template <int N, int E, int R1, int R2, int B>
__global__ void __launch_bounds__((N / E) * B, 512 / ((N / E) * B) > 0 ? 512 / ((N / E) * B) : 1) k_fresnel(const FresnelArgs p) {
    extern __shared__ float2 sm[];
    __shared__ unsigned int s_ticket[2];
    __shared__ int s_ready[2];
    pdl_trigger();                                        // (covariance / projection CTAs: one per SM, as SMs drain)
    pdl_wait();                                           // S and the zeroed counters are complete
    const unsigned int total = (unsigned int)p.T * (unsigned int)(p.RT + p.CT);
    if (threadIdx.x == 0) { s_ticket[0] = atomicAdd(p.counters, 1u); s_ready[0] = 0; }
    __syncthreads();
    int pending = -1;            // thread 0: completion counter of the previous tile, not yet published
    for (int it = 0;; ++it) {
        const unsigned int tk = s_ticket[it & 1];
        const int ready = s_ready[it & 1];
        if (tk >= total) break;
        int f, w; bool is_col;
        fresnel_decode(p, tk, f, w, is_col);
        if (!ready) {                                // rare: the dependency was not complete when the ticket was drawn
            if (threadIdx.x == 0) {
                if (pending >= 0) { red_release_add(p.counters + pending, 1u); pending = -1; }   // never wait while holding a signal
                unsigned int need;
                const unsigned int* dep = fresnel_dep(p, f, is_col, need);
                if (dep) while (ld_acquire(dep) < need) __nanosleep(32);
            }
            __syncthreads();
        }
        // the next ticket is drawn now; its value is first used in the middle of the tile, so the round trip is hidden
        unsigned int nt = 0u;
        if (threadIdx.x == 0) nt = atomicAdd(p.counters, 1u);
        auto mid = [&]() {
            if (threadIdx.x == 0) {
                // the stores of the previous tile drained long ago, so this release does not stall on them; every
                // thread's stores / scratch reads of that tile were ordered before its closing barrier (cumulativity)
                if (pending >= 0) { red_release_add(p.counters + pending, 1u); pending = -1; }
                int rdy = 1;
                if (nt < total) {
                    int nf, nw; bool ncol; unsigned int need;
                    fresnel_decode(p, nt, nf, nw, ncol);
                    const unsigned int* dep = fresnel_dep(p, nf, ncol, need);
                    if (dep) rdy = ld_acquire(dep) >= need;
                }
                s_ticket[(it + 1) & 1] = nt;
                s_ready[(it + 1) & 1] = rdy;
            }
        };
        const long long slot = (long long)(f % p.R) * p.npix;
        {
            if (!is_col) fft_tile<N, E, R1, R2, B, false, true, N>(p.rows, (long long)f * p.npix, slot, w, sm, mid);
            else         fft_tile<N, E, R1, R2, B, true, false, N>(p.cols, slot, (long long)f * p.npix, w, sm, mid);
            if constexpr (R1 == 1) __syncthreads();      // single-pass tiles have no closing barrier of their own
        }
        pending = 1 + (is_col ? p.T + f : f);
    }
    if (threadIdx.x == 0 && pending >= 0) red_release_add(p.counters + pending, 1u);
}

// ------------------------------------------------------------------------------------------------
// host side: plans, dispatch, launch
// ------------------------------------------------------------------------------------------------
static bool plan_shape(int N, int* E, int* R1, int* R2) {
    switch (N) {
        case 16:   *E = 16; *R1 = 1;  *R2 = 1;  return true;
        case 32:   *E = 32; *R1 = 1;  *R2 = 1;  return true;
        case 64:   *E = 16; *R1 = 4;  *R2 = 1;  return true;
        case 128:  *E = 16; *R1 = 8;  *R2 = 1;  return true;
        case 256:  *E = 16; *R1 = 16; *R2 = 1;  return true;
        case 512:  *E = 32; *R1 = 16; *R2 = 1;  return true;
        case 1024: *E = 32; *R1 = 32; *R2 = 1;  return true;
        case 2048: *E = 32; *R1 = 32; *R2 = 2;  return true;
        case 4096: *E = 16; *R1 = 16; *R2 = 16; return true;
    }
    return false;
}

int holo_fft_plan_init(FftPlan* p, int N) {
    p->N = N; p->tw1 = nullptr; p->tw2 = nullptr;
    if (!plan_shape(N, &p->E, &p->R1, &p->R2)) { holo_set_error("unsupported FFT length %d", N); return HOLO_ERR_ARG; }
    p->tps = N / p->E;
    const double PI = 3.14159265358979323846264338327950288;
    if (p->R1 > 1) {
        int Ns = p->E, R = p->R1;
        std::vector<float2> h((size_t)R * Ns);
        for (int r = 0; r < R; ++r)
            for (int k = 0; k < Ns; ++k) {
                double ang = -2.0 * PI * (double)r * (double)k / ((double)Ns * R);
                h[(size_t)r * Ns + k] = make_float2((float)cos(ang), (float)sin(ang));
            }
        HOLO_CUDA_OK(cudaMalloc(&p->tw1, h.size() * sizeof(float2)));
        HOLO_CUDA_OK(cudaMemcpy(p->tw1, h.data(), h.size() * sizeof(float2), cudaMemcpyHostToDevice));
    }
    if (p->R2 > 1) {
        int Ns = p->E * p->R1, R = p->R2;
        std::vector<float2> h((size_t)R * Ns);
        for (int r = 0; r < R; ++r)
            for (int k = 0; k < Ns; ++k) {
                double ang = -2.0 * PI * (double)r * (double)k / ((double)Ns * R);
                h[(size_t)r * Ns + k] = make_float2((float)cos(ang), (float)sin(ang));
            }
        HOLO_CUDA_OK(cudaMalloc(&p->tw2, h.size() * sizeof(float2)));
        HOLO_CUDA_OK(cudaMemcpy(p->tw2, h.data(), h.size() * sizeof(float2), cudaMemcpyHostToDevice));
    }
    return HOLO_OK;
}

void holo_fft_plan_free(FftPlan* p) {
    if (p->tw1) cudaFree(p->tw1);
    if (p->tw2) cudaFree(p->tw2);
    p->tw1 = p->tw2 = nullptr;
}

template <int N, int E, int R1, int R2, int B, bool COL, bool PRO, int DEFL = 0>
static int launch_fft_t(const FftArgs& a, int num_sms, int device, cudaStream_t st) {
    constexpr int threads = (N / E) * B;
    constexpr size_t smem = (R1 > 1) ? sizeof(float2) * (size_t)(N + N / E) * B : 0;
    auto kern = k_fft<N, E, R1, R2, B, COL, PRO, DEFL>;
    int blocks_per_sm = 0;
    { const int rc = holo_cached_occupancy((const void*)kern, device, threads, smem, &blocks_per_sm); if (rc) return rc; }
    int grid = a.ntiles < num_sms * blocks_per_sm ? a.ntiles : num_sms * blocks_per_sm;
    kern<<<grid, threads, smem, st>>>(a);
    HOLO_CUDA_OK(cudaGetLastError());
    return HOLO_OK;
}

// B (sequences per CTA) per length: rows aim at 256 threads; columns at >= 64-byte segments
template <bool COL, bool PRO, int DEFL = 0>
static int launch_fft(int N, const FftArgs& a, int num_sms, int device, cudaStream_t st) {
    switch (N) {
        case 16:   return launch_fft_t<16, 16, 1, 1, 16, COL, PRO, DEFL>(a, num_sms, device, st);
        case 32:   return launch_fft_t<32, 32, 1, 1, 16, COL, PRO, DEFL>(a, num_sms, device, st);
        case 64:   return launch_fft_t<64, 16, 4, 1, 16, COL, PRO, DEFL>(a, num_sms, device, st);
        case 128:  return launch_fft_t<128, 16, 8, 1, 16, COL, PRO, DEFL>(a, num_sms, device, st);
        case 256:  return launch_fft_t<256, 16, 16, 1, 16, COL, PRO, DEFL>(a, num_sms, device, st);
        case 512:  return launch_fft_t<512, 32, 16, 1, 16, COL, PRO, DEFL>(a, num_sms, device, st);
        case 1024: return launch_fft_t<1024, 32, 32, 1, 8, COL, PRO, DEFL>(a, num_sms, device, st);
        case 2048: return launch_fft_t<2048, 32, 32, 2, 4, COL, PRO, DEFL>(a, num_sms, device, st);
        case 4096: return launch_fft_t<4096, 16, 16, 16, 4, COL, PRO, DEFL>(a, num_sms, device, st);
    }
    holo_set_error("unsupported FFT length %d", N);
    return HOLO_ERR_ARG;
}

template <int N, int E, int R1, int R2, int B, int TILED = 0>
static int launch_col_energy_t(const FftArgs& a, float* out, long long npix, int nframes, int nsplit, int device, cudaStream_t st) {
    constexpr int threads = (N / E) * B;
    constexpr size_t smem = (R1 > 1) ? sizeof(float2) * (size_t)(N + N / E) * B : 0;
    auto kern = k_col_energy<N, E, R1, R2, B, TILED>;
    { const int rc = holo_ensure_smem_attr((const void*)kern, device, smem); if (rc) return rc; }
    HOLO_CUDA_OK(holo_launch_pdl(kern, dim3((unsigned)a.tiles_per_frame, (unsigned)nsplit), dim3(threads), smem, st, a, out, npix, nframes, nsplit));
    return HOLO_OK;
}
static int launch_col_energy(int N, const FftArgs& a, float* out, long long npix, int nframes, int nsplit, int device, cudaStream_t st,
                             int tiled = 0) {
    if (tiled) {
        if (N == 1024 && tiled == 8) return launch_col_energy_t<1024, 32, 32, 1, 8, 8>(a, out, npix, nframes, nsplit, device, st);
        if (N == 1024 && tiled == 16) return launch_col_energy_t<1024, 32, 32, 1, 8, 16>(a, out, npix, nframes, nsplit, device, st);
        if (N == 1024 && tiled == 32) return launch_col_energy_t<1024, 32, 32, 1, 8, 32>(a, out, npix, nframes, nsplit, device, st);
        holo_set_error("tiled column input: unsupported length %d", N);
        return HOLO_ERR_ARG;
    }
    switch (N) {
        case 16:   return launch_col_energy_t<16, 16, 1, 1, 16>(a, out, npix, nframes, nsplit, device, st);
        case 32:   return launch_col_energy_t<32, 32, 1, 1, 16>(a, out, npix, nframes, nsplit, device, st);
        case 64:   return launch_col_energy_t<64, 16, 4, 1, 16>(a, out, npix, nframes, nsplit, device, st);
        case 128:  return launch_col_energy_t<128, 16, 8, 1, 16>(a, out, npix, nframes, nsplit, device, st);
        case 256:  return launch_col_energy_t<256, 16, 16, 1, 16>(a, out, npix, nframes, nsplit, device, st);
        case 512:  return launch_col_energy_t<512, 32, 16, 1, 16>(a, out, npix, nframes, nsplit, device, st);
        case 1024: return launch_col_energy_t<1024, 32, 32, 1, 8>(a, out, npix, nframes, nsplit, device, st);
        case 2048: return launch_col_energy_t<2048, 32, 32, 2, 4>(a, out, npix, nframes, nsplit, device, st);
        case 4096: return launch_col_energy_t<4096, 16, 16, 16, 4>(a, out, npix, nframes, nsplit, device, st);
    }
    holo_set_error("unsupported FFT length %d", N);
    return HOLO_ERR_ARG;
}
#ifndef FUSED_B1024
#define FUSED_B1024 8          // sequences per CTA of the fused kernel at N = 1024 (4 = four 128-thread CTAs per SM was measured 8 % slower)
#endif
#ifndef FUSED_B2048
#define FUSED_B2048 4          // 2048: 8 (one 512-thread CTA per SM, 64-byte column segments) measured 8 % slower
#endif
static int fft_batch(int N) { return N <= 512 ? 16 : N == 1024 ? 8 : 4; }

template <int N, int E, int R1, int R2, int B>
static int launch_fresnel_t(const FresnelArgs& p, int num_sms, int device, cudaStream_t st) {
    constexpr int threads = (N / E) * B;
    constexpr size_t smem = (R1 > 1) ? sizeof(float2) * (size_t)(N + N / E) * B : 0;
    auto kern = k_fresnel<N, E, R1, R2, B>;
    int blocks_per_sm = 0;
    { const int rc = holo_cached_occupancy((const void*)kern, device, threads, smem, &blocks_per_sm); if (rc) return rc; }
    const long long total = (long long)p.T * (p.RT + p.CT);
    long long grid = (long long)num_sms * blocks_per_sm;      // one wave of persistent CTAs
    if (grid > total) grid = total;
    HOLO_CUDA_OK(holo_launch_pdl(kern, dim3((unsigned)grid), dim3(threads), smem, st, p));
    HOLO_CUDA_OK(cudaGetLastError());
    return HOLO_OK;
}

static int launch_fresnel_fused(int N, const FresnelArgs& p, int num_sms, int device, cudaStream_t st) {
    switch (N) {
        case 16:   return launch_fresnel_t<16, 16, 1, 1, 16>(p, num_sms, device, st);
        case 32:   return launch_fresnel_t<32, 32, 1, 1, 16>(p, num_sms, device, st);
        case 64:   return launch_fresnel_t<64, 16, 4, 1, 16>(p, num_sms, device, st);
        case 128:  return launch_fresnel_t<128, 16, 8, 1, 16>(p, num_sms, device, st);
        case 256:  return launch_fresnel_t<256, 16, 16, 1, 16>(p, num_sms, device, st);
        case 512:  return launch_fresnel_t<512, 32, 16, 1, 16>(p, num_sms, device, st);
        case 1024: return launch_fresnel_t<1024, 32, 32, 1, FUSED_B1024>(p, num_sms, device, st);
        case 2048: return launch_fresnel_t<2048, 32, 32, 2, FUSED_B2048>(p, num_sms, device, st);
        case 4096: return launch_fresnel_t<4096, 16, 16, 16, 4>(p, num_sms, device, st);
    }
    holo_set_error("unsupported FFT length %d", N);
    return HOLO_ERR_ARG;
}

static bool use_fused(const holo_ctx* c) {
    return c->nx == c->ny && c->tune[HOLO_TUNE_FFT_PERSISTENT] && c->scratch_frames >= 2 && 2 * c->T + 1 <= 256;
}

// Fresnel stage as two streaming kernels (packed row pass -> row-pass output of the whole stack in c->rowout -> column pass)
// instead of the fused persistent kernel: 2048 x 2048 (any frame count), and 1024 x 1024 for an even frame count of at
// least 16 (shorter runs -- the strides of holo_push -- are faster in the fused kernel, whose ring stays in L2)
static bool use_packed_pair(const holo_ctx* c, int nproc) {
    if (!c->rowout) return false;
    if (c->nx == 2048 && c->ny == 2048) return c->tune[HOLO_TUNE_COLS2048] != 0;
    if (c->nx == 1024 && c->ny == 1024) return c->tune[HOLO_TUNE_PACKED1024] != 0 && (c->T % 2) == 0 && (nproc % 2) == 0 && nproc >= 16;
    return false;
}

bool holo_fresnel_is_packed(const holo_ctx* c) { return use_packed_pair(c, c->T); }

int holo_fresnel_launch_count(holo_ctx* c) {
    if (use_packed_pair(c, c->T)) return 3;
    if (use_fused(c)) return 2;
    int g = c->scratch_frames;
    int groups = (c->T + g - 1) / g;
    return 1 + 2 * groups;
}

// A0 alone (also zeroes the counters of the fused Fresnel kernel)
int holo_launch_sum(holo_ctx* c, const uint16_t* frames, cudaStream_t st) {
    long long nvec = c->npix >> 3;
    int threads = 256;
    long long want = (nvec + threads - 1) / threads;
    int grid = (int)(want < (long long)c->num_sms * 8 ? want : (long long)c->num_sms * 8);
    HoloProf prof(c, HOLO_K_SUM, st);
    k_frame_sum<<<grid, threads, 0, st>>>(frames, c->sum, c->npix, c->T, c->counters);
    HOLO_CUDA_OK(cudaGetLastError());
    return HOLO_OK;
}

// with_sum = false: c->sum already holds the reference sum image S (d = (T I - S)/T); nproc = number of frames to
// transform (frames[0..nproc) -> H[0..nproc)), default all T
int holo_launch_fresnel(holo_ctx* c, const uint16_t* frames, float2* H, cudaStream_t st, bool with_sum, int nproc, bool counters_zeroed) {
    if (nproc < 0) nproc = c->T;
    if (with_sum) { const int rc = holo_launch_sum(c, frames, st); if (rc) return rc; }
    else if (!counters_zeroed && use_fused(c) && !use_packed_pair(c, nproc))
        HOLO_CUDA_OK(cudaMemsetAsync(c->counters, 0, (2 * c->T + 1) * sizeof(unsigned int), st));
    if (use_packed_pair(c, nproc)) {
        // the row ticket: zeroed by the sum kernels (k_frame_sum, k_sum_gram) where one of them ran just before
        if (!with_sum && !counters_zeroed) HOLO_CUDA_OK(cudaMemsetAsync(c->counters + 1001, 0, sizeof(unsigned int), st));
        if (c->nx == 2048) {
            // 2048 x 2048: the packed row pass (radix-2 decimation in frequency + a pair of 1024-point transforms) and the
            // packed column pass, the row-pass output of the stack going through HBM: 1.8 vs 2.4 ms for the fused three-pass kernel
            int rc = holo_launch_rows2(c, frames, c->rowout, 0, st, nproc);
            if (rc) return rc;
            return holo_launch_cols2048_store(c, c->rowout, H, nproc, st);
        }
        // 1024 x 1024: the packed row pass of frame pairs stores its output in column blocks of 8 columns, the column pass
        // reads one contiguous 64 KB block per tile: both kernels stream at ~80 % of the HBM peak on their DRAM traffic
        // (871 MB with the intermediate) and take 168 us together; the fused kernel keeps the intermediate in L2 (438 MB
        // of DRAM traffic) but is bound by the dependency stalls of its tile pipeline: 197 us
        int rc = holo_launch_rows2(c, frames, c->rowout, 0, st, nproc, 8);
        if (rc) return rc;
        FftArgs b{};
        b.in = c->rowout; b.out = H;
        b.tw1 = c->py.tw1; b.tw2 = c->py.tw2;
        b.in_fstride = c->npix; b.out_fstride = c->npix;
        b.ld = c->nx; b.nseq = c->nx;
        b.tiles_per_frame = c->nx / 8;
        b.ntiles = nproc * b.tiles_per_frame;
        b.T = c->T;
        constexpr size_t smem = sizeof(float2) * (size_t)(1024 + 32) * 8;
        auto kern = k_cols_tiled<1024, 32, 32, 1, 8>;
        int blocks_per_sm = 0;
        if ((rc = holo_cached_occupancy((const void*)kern, c->device, 256, smem, &blocks_per_sm))) return rc;
        const int sms = c->num_sms - c->fresnel_sm_reserve;    // (mode 2: one SM for the side-stream eigensolver)
        const int grid = b.ntiles < sms * blocks_per_sm ? b.ntiles : sms * blocks_per_sm;
        HoloProf prof(c, HOLO_K_FFT_COLS, st);
        HOLO_CUDA_OK(holo_launch_pdl(kern, dim3(grid), dim3(256), smem, st, b));
        return HOLO_OK;
    }
    if (use_fused(c)) {
        FresnelArgs p{};
        const int Bq = c->nx == 1024 ? FUSED_B1024 : c->nx == 2048 ? FUSED_B2048 : fft_batch(c->nx);
        FftArgs& a = p.rows;
        a.frames = frames; a.sum = c->sum; a.qx = c->qxs; a.qy = c->qy; a.in = nullptr; a.out = c->scratch;
        a.tw1 = c->px.tw1; a.tw2 = c->px.tw2; a.ld = c->nx; a.nseq = c->ny; a.T = c->T;
        FftArgs& b = p.cols;
        b.in = c->scratch; b.out = H; b.tw1 = c->py.tw1; b.tw2 = c->py.tw2; b.ld = c->nx; b.nseq = c->nx; b.T = c->T;
        p.counters = c->counters; p.npix = c->npix; p.T = nproc; p.R = c->scratch_frames;
        p.L = c->tune[HOLO_TUNE_FFT_LAG] > 0 ? c->tune[HOLO_TUNE_FFT_LAG] : p.R / 2;
        if (p.L > p.R - 1) p.L = p.R - 1;
        if (p.L > p.T) p.L = p.T;
        if (p.L < 1) p.L = 1;
        p.RT = c->ny / Bq; p.CT = c->nx / Bq;
        HoloProf prof(c, HOLO_K_FFT_ROWS, st);
        // fresnel_sm_reserve: SMs left to a side-stream kernel that must run UNDER this persistent launch (mode 2: the
        // eigensolver of the same stack; a persistent kernel that fills every SM would make it wait for the end)
        return launch_fresnel_fused(c->nx, p, c->num_sms - c->fresnel_sm_reserve, c->device, st);
    }
    // A1 + A2, frame groups so that the row->column intermediate stays in L2
    const int G = c->scratch_frames;
    for (int f0 = 0; f0 < nproc; f0 += G) {
        const int nf = (nproc - f0 < G) ? nproc - f0 : G;
        FftArgs a{};
        a.frames = frames + (long long)f0 * c->npix;
        a.sum = c->sum; a.qx = c->qxs; a.qy = c->qy;
        a.in = nullptr; a.out = c->scratch;
        a.tw1 = c->px.tw1; a.tw2 = c->px.tw2;
        a.in_fstride = c->npix; a.out_fstride = c->npix;
        a.ld = c->nx; a.nseq = c->ny;
        a.tiles_per_frame = c->ny / fft_batch(c->nx);
        a.ntiles = nf * a.tiles_per_frame;
        a.T = c->T;
        int rc;
        { HoloProf prof(c, HOLO_K_FFT_ROWS, st); rc = launch_fft<false, true>(c->nx, a, c->num_sms, c->device, st); }
        if (rc) return rc;
        FftArgs b{};
        b.in = c->scratch; b.out = H + (long long)f0 * c->npix;
        b.tw1 = c->py.tw1; b.tw2 = c->py.tw2;
        b.in_fstride = c->npix; b.out_fstride = c->npix;
        b.ld = c->nx; b.nseq = c->nx;
        b.tiles_per_frame = c->nx / fft_batch(c->ny);
        b.ntiles = nf * b.tiles_per_frame;
        b.T = c->T;
        { HoloProf prof(c, HOLO_K_FFT_COLS, st); rc = launch_fft<true, false>(c->ny, b, c->num_sms, c->device, st); }
        if (rc) return rc;
    }
    return HOLO_OK;
}

// ------------------------------------------------------------------------------------------------
// Mode 3 (SURVEY.md 8(f)-2 stage 2): the image without the hologram stack.  Needs S = sum_t I_t in c->sum and the
// eigenvectors V (real: the covariance of the raw frames is real symmetric, R21).
//   1. k_deflate_images: eT_k = sum_t (T I_t - S) V_tk for the rejected components k (at most 4)
//   2. row pass of all T frames with the deflation in the prologue -> G = row transform of q (d_t - sum_k e_k V_tk)
//      (complex64 [T][ny][nx] in c->H: the only large intermediate, written and read once)
//   3. k_col_energy: column transform reduced to sum_t |.|^2, frame splits -> k_sum_partial_images
// ------------------------------------------------------------------------------------------------
int holo_mode3_splits(const holo_ctx* c, int nframes) {
    if (c->tune[HOLO_TUNE_COLS2048] && holo_cols2048_supported(c)) return nframes >= 4 ? 4 : 1;   // packed kernel: (tile, quarter of the frames) units
    const int ct = c->nx / fft_batch(c->ny);
    int ns = (2 * c->num_sms) / (ct > 0 ? ct : 1);
    if (ns < 1) ns = 1;
    if (ns > nframes) ns = nframes;
    if (ns > 8) ns = 8;
    return ns;
}

// frame basis (T transforms, at most 4 components removed in the raw domain) or eigen basis (nS transforms of the kept
// components' raw-domain images): the cheaper one that is possible
bool holo_mode3_eigen_form(const holo_ctx* c, int k_lo, int k_hi) {
    const int T = c->T, nS = k_hi - k_lo + 1, ndefl = T - nS;
    return ndefl > 4 || 4 * nS <= 3 * T;
}

int holo_launch_energy_image(holo_ctx* c, const uint16_t* frames, const float2* V, int k_lo, int k_hi, float* image, cudaStream_t st) {
    const int T = c->T;
    const int n0 = k_lo - 1, n1 = T - k_hi, ndefl = n0 + n1, nS = k_hi - k_lo + 1;
    const bool eigen = holo_mode3_eigen_form(c, k_lo, k_hi);
    if (eigen && !c->eig_img) { holo_set_error("internal: eigen-image workspace missing (holo_set_mode / holo_set_range allocate it)"); return HOLO_ERR_STATE; }
    int rc = HOLO_OK;
    const int nframes = eigen ? nS : T;
    // row ticket (k_sum_gram may run on another stream).  First in the chain: the kernels below follow one another as
    // programmatic dependent launches (deflation images -> row pass -> column pass -> sum of the partial images)
    HOLO_CUDA_OK(cudaMemsetAsync(c->counters + 1001, 0, sizeof(unsigned int), st));
    if (eigen) {
        HoloProf prof(c, HOLO_K_SUM, st);
        const int px = T <= 32 ? 4 : 2;
        const long long nvec = c->npix / px;
        long long want = (nvec + 127) / 128;
        const int grid = (int)(want < (long long)c->num_sms * 8 ? want : (long long)c->num_sms * 8);
        if (T <= 32) k_eigen_images<32, 4><<<grid, 128, (size_t)nS * 32 * sizeof(float), st>>>(frames, c->sum, V, c->npix, T, k_lo - 1, nS, c->eig_img);
        else         k_eigen_images<64, 2><<<grid, 128, (size_t)nS * 64 * sizeof(float), st>>>(frames, c->sum, V, c->npix, T, k_lo - 1, nS, c->eig_img);
        HOLO_CUDA_OK(cudaGetLastError());
    } else if (ndefl > 0) {
        HoloProf prof(c, HOLO_K_SUM, st);
        const long long nvec = c->npix >> 3;
        long long want = (nvec + 255) / 256;
        const int grid = (int)(want < (long long)c->num_sms * 8 ? want : (long long)c->num_sms * 8);
        switch (ndefl) {
            case 1: k_deflate_images<1><<<grid, 256, 0, st>>>(frames, c->sum, V, c->npix, T, 0, n0, k_hi, c->defl_img, c->defl_coef); break;
            case 2: k_deflate_images<2><<<grid, 256, 0, st>>>(frames, c->sum, V, c->npix, T, 0, n0, k_hi, c->defl_img, c->defl_coef); break;
            case 3: k_deflate_images<3><<<grid, 256, 0, st>>>(frames, c->sum, V, c->npix, T, 0, n0, k_hi, c->defl_img, c->defl_coef); break;
            default: k_deflate_images<4><<<grid, 256, 0, st>>>(frames, c->sum, V, c->npix, T, 0, n0, k_hi, c->defl_img, c->defl_coef); break;
        }
        HOLO_CUDA_OK(cudaGetLastError());
    }
    FftArgs a{};
    a.frames = frames; a.sum = c->sum; a.qx = c->qxs; a.qy = c->qy; a.in = nullptr; a.out = c->H;
    a.tw1 = c->px.tw1; a.tw2 = c->px.tw2;
    a.in_fstride = c->npix; a.out_fstride = c->npix;
    a.ld = c->nx; a.nseq = c->ny;
    a.tiles_per_frame = c->ny / fft_batch(c->nx);
    a.ntiles = nframes * a.tiles_per_frame;
    a.T = T;
    a.defl_img = c->defl_img; a.defl_coef = c->defl_coef; a.ndefl = ndefl;
    a.eimg = c->eig_img;
    a.ticket = c->counters + 1001;
    // the packed row pass can write its output column tile by column tile (the layout is private to this function): the
    // column pass then reads one contiguous 64 KB block per tile and frame instead of 1024 segments of 64 bytes
    const bool rows2 = !eigen && c->tune[HOLO_TUNE_ROWS2] && holo_rows2_supported(c);
    const int tiled = rows2 && c->nx == 1024 && c->ny == 1024 ? c->tune[HOLO_TUNE_TILED_G] : 0;
    if (eigen) { HoloProf prof(c, HOLO_K_FFT_ROWS, st); rc = launch_fft<false, true, 2>(c->nx, a, c->num_sms, c->device, st); }
    else if (rows2) rc = holo_launch_rows2(c, frames, c->H, ndefl, st, 0, tiled);
    else
    { HoloProf prof(c, HOLO_K_FFT_ROWS, st);
      rc = ndefl ? launch_fft<false, true, 1>(c->nx, a, c->num_sms, c->device, st) : launch_fft<false, true, 0>(c->nx, a, c->num_sms, c->device, st); }
    if (rc) return rc;
    FftArgs b{};
    b.in = c->H; b.out = nullptr;
    b.tw1 = c->py.tw1; b.tw2 = c->py.tw2;
    b.in_fstride = c->npix; b.out_fstride = 0;
    b.ld = c->nx; b.nseq = c->nx;
    b.tiles_per_frame = c->nx / fft_batch(c->ny);
    b.ntiles = b.tiles_per_frame;
    b.T = T;
    const int ns = holo_mode3_splits(c, nframes);
    if (c->tune[HOLO_TUNE_COLS2048] && holo_cols2048_supported(c)) {
        rc = holo_launch_cols2048(c, c->H, ns > 1 ? c->energy_parts : image, nframes, ns, st);
    } else {
        HoloProf prof(c, HOLO_K_FFT_COLS, st);
        rc = launch_col_energy(c->ny, b, ns > 1 ? c->energy_parts : image, c->npix, nframes, ns, c->device, st, tiled);
    }
    if (rc) return rc;
    if (ns > 1) {
        HoloProf prof(c, HOLO_K_PROJECT, st);
        const long long want = ((c->npix >> 2) + 255) / 256;
        HOLO_CUDA_OK(holo_launch_pdl(k_sum_partial_images, dim3((unsigned)(want < 8ll * c->num_sms ? want : 8ll * c->num_sms)), dim3(256), 0, st,
                                     (const float*)c->energy_parts, ns, c->npix, image));
    }
    return HOLO_OK;
}
