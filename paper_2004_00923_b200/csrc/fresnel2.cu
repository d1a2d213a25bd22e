// fresnel2.cu -- packed two-sequence FFT building blocks and the mode-3 row pass built on them (1024-point rows):
//   G_t = row transform of (d_t - sum_k e_k V_tk) * exp(+i pi (x^2+y^2)/(lambda z))     (Eq. 1)
// TWO sequences per thread in structure-of-arrays register pairs (re_a, re_b), (im_a, im_b): every butterfly of the
// radix-32 networks is a packed FADD2 / FFMA2 on both sequences (same twiddle), i.e. half the FP32 issue slots of the
// scalar form; 32 elements of each sequence per thread, so ONE WARP owns a pair of 1024-point sequences: pass 0
// (radix 32), one exchange through a warp-private, XOR-skewed shared-memory region (16-byte accesses, conflict free),
// pass 1 (radix 32); only __syncwarp inside a transform.
// (Round 2 also built a fused persistent Fresnel kernel on these blocks -- packed row pairs, TMA-staged column tiles in
// a super-tile pipeline -- which was correct and 12 % slower than k_fresnel, 220 vs 197 us; it is not kept.)
#include "holo_internal.cuh"
#include "fft_reg.cuh"
#include "tma.cuh"

namespace {

constexpr int F2N = 1024;                 // sequence length (rows and columns)
constexpr int F2_TILE = 65536;            // bytes of the exchange region of four warps: 4 x 2 sequences x 1024 x 8 B
struct cpk { float2 re, im; };            // one complex value of each of the two sequences (.x: sequence a, .y: b)

__device__ __forceinline__ float2 pneg(float2 a) { return make_float2(-a.x, -a.y); }
__device__ __forceinline__ float2 padd(float2 a, float2 b) { return __fadd2_rn(a, b); }
__device__ __forceinline__ float2 psub(float2 a, float2 b) { return __fadd2_rn(a, pneg(b)); }
__device__ __forceinline__ float2 pfma(float c, float2 x, float2 y) { return __ffma2_rn(make_float2(c, c), x, y); }

// (tr, ti) and sc with  w b = sc (tr, ti)  for w = exp(-2 pi i E32 / 32), 0 < E32 < 16, E32 != 8 (see bfly_dit)
template <int E32> __device__ __forceinline__ void twid_t(const cpk& b, float2& tr, float2& ti, float& sc) {
    constexpr double wr = cos32d(E32), wi = -sin32d(E32);
    constexpr bool tanform = (wr < 0 ? -wr : wr) >= (wi < 0 ? -wi : wi);
    if constexpr (E32 == 4) { tr = padd(b.re, b.im); ti = psub(b.im, b.re); sc = (float)wr; }
    else if constexpr (E32 == 12) { tr = psub(b.re, b.im); ti = padd(b.im, b.re); sc = (float)wr; }
    else if constexpr (tanform) {
        constexpr float c = (float)(wi / wr);
        tr = pfma(-c, b.im, b.re); ti = pfma(c, b.re, b.im); sc = (float)wr;
    } else {
        constexpr float c = (float)(wr / wi);
        tr = pfma(c, b.re, pneg(b.im)); ti = pfma(c, b.im, b.re); sc = (float)wi;
    }
}

// packed DIT butterfly on both sequences: (a, b) <- (a + w b, a - w b)
template <int E32> __device__ __forceinline__ void bfly2(cpk& a, cpk& b) {
    if constexpr (E32 == 0) {
        const cpk t = b;
        b.re = psub(a.re, t.re); b.im = psub(a.im, t.im);
        a.re = padd(a.re, t.re); a.im = padd(a.im, t.im);
    } else if constexpr (E32 == 8) {                      // w = -i: w b = (b_im, -b_re)
        const cpk t = b;
        b.re = psub(a.re, t.im); b.im = padd(a.im, t.re);
        a.re = padd(a.re, t.im); a.im = psub(a.im, t.re);
    } else {
        float2 tr, ti; float sc;
        twid_t<E32>(b, tr, ti, sc);
        b.re = pfma(-sc, tr, a.re); b.im = pfma(-sc, ti, a.im);
        a.re = pfma(sc, tr, a.re); a.im = pfma(sc, ti, a.im);
    }
}

// the same butterfly with array-of-structures results (re_a, im_a, re_b, im_b): the last stage of a tile
template <int E32> __device__ __forceinline__ void bfly2_to_aos(const cpk& a, const cpk& b, float4& oa, float4& ob) {
    if constexpr (E32 == 0) {
        oa = make_float4(a.re.x + b.re.x, a.im.x + b.im.x, a.re.y + b.re.y, a.im.y + b.im.y);
        ob = make_float4(a.re.x - b.re.x, a.im.x - b.im.x, a.re.y - b.re.y, a.im.y - b.im.y);
    } else if constexpr (E32 == 8) {
        oa = make_float4(a.re.x + b.im.x, a.im.x - b.re.x, a.re.y + b.im.y, a.im.y - b.re.y);
        ob = make_float4(a.re.x - b.im.x, a.im.x + b.re.x, a.re.y - b.im.y, a.im.y + b.re.y);
    } else {
        float2 tr, ti; float sc;
        twid_t<E32>(b, tr, ti, sc);
        oa = make_float4(fmaf(sc, tr.x, a.re.x), fmaf(sc, ti.x, a.im.x), fmaf(sc, tr.y, a.re.y), fmaf(sc, ti.y, a.im.y));
        ob = make_float4(fmaf(-sc, tr.x, a.re.x), fmaf(-sc, ti.x, a.im.x), fmaf(-sc, tr.y, a.re.y), fmaf(-sc, ti.y, a.im.y));
    }
}

// stages S0 .. S1-1 of the radix-32 DIT network on v[0..32) (natural-order input; X[k] = v[brev<32>(k)] after stage 4)
template <int S, int G, int M> struct P2M {
    static __device__ __forceinline__ void run(cpk* v) {
        constexpr int span = 32 >> (S + 1);
        constexpr int e32 = brev<(1 << S)>(G) * (16 >> S);
        bfly2<e32>(v[2 * span * G + M], v[2 * span * G + M + span]);
        if constexpr (M + 1 < span) P2M<S, G, M + 1>::run(v);
    }
};
template <int S, int G> struct P2G {
    static __device__ __forceinline__ void run(cpk* v) {
        P2M<S, G, 0>::run(v);
        if constexpr (G + 1 < (1 << S)) P2G<S, G + 1>::run(v);
    }
};
template <int S0, int S1> struct P2S {
    static __device__ __forceinline__ void run(cpk* v) {
        if constexpr (S0 < S1) { P2G<S0, 0>::run(v); P2S<S0 + 1, S1>::run(v); }
    }
};
// stage 4 (pairs (2g, 2g+1), twiddle brev<16>(g)) with AoS results: o[p] = value of register slot p
template <int G> struct P2Last {
    static __device__ __forceinline__ void run(const cpk* v, float4* o) {
        bfly2_to_aos<brev<16>(G)>(v[2 * G], v[2 * G + 1], o[2 * G], o[2 * G + 1]);
        if constexpr (G + 1 < 16) P2Last<G + 1>::run(v, o);
    }
};

__device__ __forceinline__ float4 lds128(uint32_t addr) {
    float4 v;
    asm volatile("ld.shared.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(addr));
    return v;
}
__device__ __forceinline__ void sts128(uint32_t addr, float4 v) {
    asm volatile("st.shared.v4.f32 [%0], {%1,%2,%3,%4};" ::"r"(addr), "f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w) : "memory");
}
// ---- exchange layout of one warp inside a tile buffer --------------------------------------------------------
// The warp owns the 16-byte chunk `wg` of every 64-byte row n of the buffer (1024 slots), stored at chunk position
// wg ^ ((n >> 1) & 3) -- the TMA unit's SWIZZLE_64B pattern, so that the rows it delivers (n = row of the frame) and
// the rows it stores are addressed by the same formula.  Between the passes element (j, k) [source lane j, output k of
// pass 0] lives in slot n = 32 k + (j ^ (k & 7)): lanes j (writes) and lanes k (reads) then both hit eight different
// 16-byte bank groups per quarter warp.  All addresses are  per-lane base (8 variants) + immediate.
struct XAddr {
    uint32_t wr[8];   // write side (lane = j): variant k & 7, + 2048 k
    uint32_t rd[8];   // read side (lane = k): variant r & 7, + 512 (r >> 3)
    uint32_t nat;     // natural rows n = lane + 32 m: + 2048 m
};
__device__ __forceinline__ XAddr make_xaddr(uint32_t buf, int wg, int lane) {
    XAddr x;
    const uint32_t cl = (uint32_t)(wg ^ ((lane >> 1) & 3));
    const uint32_t basel = (uint32_t)lane * 64u + (cl << 4);
    x.nat = buf + basel;
#pragma unroll
    for (int c = 0; c < 8; ++c) {
        const uint32_t K = (uint32_t)c * 64u + (uint32_t)(((c >> 1) & 3) << 4);
        x.wr[c] = buf + (basel ^ K);                                                  // slot 32 k + (lane ^ c), k & 7 = c
        x.rd[c] = buf + (uint32_t)lane * 2048u + (K ^ ((uint32_t)(lane & 7) * 64u + (cl << 4)));   // slot 32 lane + (r ^ (lane & 7)), r & 7 = c
    }
    return x;
}

// pass 0 results -> exchange (SoA float4: re_a, re_b, im_a, im_b)
__device__ __forceinline__ void exchange_write(const XAddr& x, const cpk* v) {
#pragma unroll
    for (int k = 0; k < 32; ++k) {
        const cpk e = v[brev<32>(k)];
        sts128(x.wr[k & 7] + 2048u * k, make_float4(e.re.x, e.re.y, e.im.x, e.im.y));
    }
}
// exchange -> pass 1 inputs of lane b (element r came from lane r), times the inter-pass twiddle W_1024^{r b}
__device__ __forceinline__ void exchange_read_twiddle(const XAddr& x, cpk* v, const float2* tw_s, int lane) {
#pragma unroll
    for (int r = 0; r < 32; ++r) {
        const float4 e = lds128(x.rd[r & 7] + 512u * (r >> 3));
        v[r].re = make_float2(e.x, e.y);
        v[r].im = make_float2(e.z, e.w);
    }
#pragma unroll
    for (int r = 1; r < 32; ++r) {
        const float2 w = tw_s[r * 32 + lane];
        const float2 re = pfma(w.x, v[r].re, pneg(__fmul2_rn(make_float2(w.y, w.y), v[r].im)));
        const float2 im = pfma(w.x, v[r].im, __fmul2_rn(make_float2(w.y, w.y), v[r].re));
        v[r].re = re; v[r].im = im;
    }
}

// ------------------------------------------------------------------------------------------------
// Mode 3 row pass, packed form (1024-point rows): one warp transforms row y of TWO consecutive frames (f, f + 1) at once.
// The frame sum S, the deflation images e_k and the chirp of the row are loaded once for both, every butterfly is a
// packed FADD2 / FFMA2 on the pair, the exchange uses 16-byte accesses: about 60 % of the instructions and of the L1
// traffic of the scalar row kernel (k_fft), which ncu shows bound by instruction issue (58 %) and the L1 pipe (72 %).
// Warps are autonomous (row pairs drawn from a ticket, warp-private exchange slice, no CTA-wide step).
// ------------------------------------------------------------------------------------------------
struct R2Args {
    const uint16_t* frames;   // [T][ny][nx]
    const uint32_t* sum;      // S = sum_t I_t
    const float2* qxs;        // chirp along x, scaled by 1/T
    const float2* qy;
    const float2* tw;         // [32][32] inter-pass twiddles of the 1024-point transform
    const float2* tw2048;     // NX = 2048: exp(-2 pi i n / 2048), n < 1024
    const float* defl_img;    // [ndefl][ny][nx]  eT_k
    const float* defl_coef;   // [T][ndefl]
    float2* out;              // [T][ny][nx] row-pass output
    unsigned int* ticket;     // zeroed by an earlier operation of the stream
    int T, ndefl, ny;
    int nframes;              // frames to transform (T, or fewer: sliding window); T itself enters d = T I - S
    int tile_w;               // NX = 1024: 0 = row-major output; w = output stored [frame][x / w][y][x % w] (w divides 32)
};

constexpr int R2_WARPS = 12;
template <int NX> constexpr int r2_smem() { return 1024 + (R2_WARPS / 4) * F2_TILE + F2N * 8 + NX * 8 + (NX == 2048 ? F2N * 8 : 0); }

// NX = 1024: a warp transforms row y of the two frames (f, f + 1): the packed pair is (frame f, frame f + 1).
// NX = 2048: a warp transforms ONE row of 2048 points: a radix-2 decimation-in-frequency step in the prologue,
//   y0(n) = x(n) + x(n + 1024),  y1(n) = (x(n) - x(n + 1024)) W_2048^n,   X(2k) = FFT1024[y0](k), X(2k + 1) = FFT1024[y1](k),
// makes the packed pair (y0, y1); the two results of a register slot are adjacent outputs: one 16-byte store.
template <int NX>
__global__ void __launch_bounds__(R2_WARPS * 32, 1) k_rows2(const R2Args a) {
    extern __shared__ unsigned char smraw_[];
    const uint32_t s0 = smem_u32(smraw_);
    const uint32_t pad = (1024u - (s0 & 1023u)) & 1023u;
    unsigned char* base = smraw_ + pad;
    const uint32_t bufs = s0 + pad;
    float2* tw_s = reinterpret_cast<float2*>(base + (R2_WARPS / 4) * F2_TILE);
    float2* qx_s = tw_s + F2N;
    float2* w2_s = qx_s + NX;                                  // NX = 2048 only
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    for (int i = tid; i < F2N; i += R2_WARPS * 32) tw_s[i] = a.tw[i];
    for (int i = tid; i < NX; i += R2_WARPS * 32) qx_s[i] = a.qxs[i];
    if constexpr (NX == 2048) for (int i = tid; i < F2N; i += R2_WARPS * 32) w2_s[i] = a.tw2048[i];
    // (no early trigger here: column CTAs made resident while this kernel drains pile up three deep on the SMs that finish
    //  first and leave the others empty: 224 vs 206 us per stack)
    pdl_wait();                                                // the tables above never change; everything below depends on earlier kernels
    __syncthreads();
    const uint32_t buf = bufs + (uint32_t)(warp >> 2) * F2_TILE;
    const XAddr xa = make_xaddr(buf, warp & 3, lane);
    const long long npix = (long long)NX * a.ny;
    const unsigned int ntasks = NX == 1024 ? (unsigned int)(a.nframes / 2) * (unsigned int)a.ny : (unsigned int)a.nframes * (unsigned int)a.ny;
    const float Tf = (float)a.T;
    // tickets are drawn two tasks ahead (the atomic's round trip is hidden) and the frame rows of the NEXT task are pulled
    // into L2 while the current one computes (ncu: 14 % of the warp time waited for the ticket, 30 % for the loads)
    unsigned int tk0 = 0u, tk1 = 0u;
    if (lane == 0) { tk0 = atomicAdd(a.ticket, 1u); tk1 = atomicAdd(a.ticket, 1u); }
    tk0 = __shfl_sync(0xffffffffu, tk0, 0); tk1 = __shfl_sync(0xffffffffu, tk1, 0);
    for (;;) {
        const unsigned int tk = tk0;
        if (tk >= ntasks) break;
        unsigned int tk2 = 0u;
        if (lane == 0) tk2 = atomicAdd(a.ticket, 1u);
        if (tk1 < ntasks) {
            const int f1 = NX == 1024 ? 2 * (int)(tk1 / (unsigned int)a.ny) : (int)(tk1 % (unsigned int)a.nframes);
            const int y1 = NX == 1024 ? (int)(tk1 % (unsigned int)a.ny) : (int)(tk1 / (unsigned int)a.nframes);
            const uint16_t* pf = NX == 1024 ? a.frames + (long long)(f1 + (lane >> 4)) * npix + (long long)y1 * NX + (lane & 15) * 64
                                            : a.frames + (long long)f1 * npix + (long long)y1 * NX + lane * 64;
            asm volatile("prefetch.global.L2 [%0];" ::"l"(pf));
        }
        // task order.  NX = 1024: row-minor (consecutive tickets = consecutive rows of a frame pair: the frames are written one after
        // the other and the column pass finds the last ones in L2).  NX = 2048: FRAME-minor (consecutive tickets = the same row of
        // consecutive frames): the twelve warps of a CTA then share the row of S and of the deflation images through L1 instead
        // of fetching 8 + 8 n_rej KB per task from L2 (mode 3 at 2048^2 x 64: row pass 965 -> 686 us; mode 1: 622 -> 580 us; at
        // 1024 points the same order measured 1 - 2 us slower in both passes)
        const int f = NX == 1024 ? 2 * (int)(tk / (unsigned int)a.ny) : (int)(tk % (unsigned int)a.nframes);
        const int y = NX == 1024 ? (int)(tk % (unsigned int)a.ny) : (int)(tk / (unsigned int)a.nframes);
        const uint16_t* Ia = a.frames + (long long)f * npix + (long long)y * NX + lane;
        const uint32_t* Sp = a.sum + (long long)y * NX + lane;
        const float2 qyv = __ldg(a.qy + y);
        cpk v[32];
        // second element of the pair: the same position of frame f + 1 (NX = 1024) / position n + 1024 of the same row
        const long long poff = NX == 1024 ? npix : 1024;
        // d = T I - S exactly (integers below 2^23)
#pragma unroll
        for (int m = 0; m < 32; ++m) {
            const float ia = (float)__ldg(Ia + 32 * m), ib = (float)__ldg(Ia + poff + 32 * m);
            const float sa = (float)__ldg(Sp + 32 * m);
            const float sb = NX == 1024 ? sa : (float)__ldg(Sp + 1024 + 32 * m);
            v[m].re = make_float2(fmaf(Tf, ia, -sa), fmaf(Tf, ib, -sb));
        }
        const float* ep = a.defl_img + (long long)y * NX + lane;
        for (int kk = 0; kk < a.ndefl; ++kk) {
            const float ca = -__ldg(a.defl_coef + f * a.ndefl + kk);
            const float2 cf = make_float2(ca, NX == 1024 ? -__ldg(a.defl_coef + (f + 1) * a.ndefl + kk) : ca);
            float e[32], e2[NX == 1024 ? 1 : 32];
#pragma unroll
            for (int m = 0; m < 32; ++m) { e[m] = __ldg(ep + 32 * m); if constexpr (NX == 2048) e2[m] = __ldg(ep + 1024 + 32 * m); }
#pragma unroll
            for (int m = 0; m < 32; ++m) v[m].re = __ffma2_rn(make_float2(e[m], NX == 1024 ? e[m] : e2[m]), cf, v[m].re);
            ep += npix;
        }
        if constexpr (NX == 1024) {
#pragma unroll
            for (int m = 0; m < 32; ++m) {
                const float2 q = cmul(qx_s[lane + 32 * m], qyv);
                const float2 d = v[m].re;
                v[m].re = __fmul2_rn(d, make_float2(q.x, q.x));
                v[m].im = __fmul2_rn(d, make_float2(q.y, q.y));
            }
        } else {
#pragma unroll
            for (int m = 0; m < 32; ++m) {
                const int n = lane + 32 * m;
                const float2 qa = cmul(qx_s[n], qyv), qb = cmul(qx_s[n + 1024], qyv);
                const float2 d = v[m].re;
                const float2 xa2 = make_float2(d.x * qa.x, d.x * qa.y), xb2 = make_float2(d.y * qb.x, d.y * qb.y);
                const float2 y0 = make_float2(xa2.x + xb2.x, xa2.y + xb2.y);
                const float2 y1 = cmul(make_float2(xa2.x - xb2.x, xa2.y - xb2.y), w2_s[n]);
                v[m].re = make_float2(y0.x, y1.x);
                v[m].im = make_float2(y0.y, y1.y);
            }
        }
        P2S<0, 5>::run(v);
        exchange_write(xa, v);
        __syncwarp();
        exchange_read_twiddle(xa, v, tw_s, lane);
        __syncwarp();
        P2S<0, 4>::run(v);
        float4 o[32];
        P2Last<0>::run(v, o);
        if constexpr (NX == 1024) {
            // X[lane + 32 kk] of frame f in (o.x, o.y), of frame f + 1 in (o.z, o.w); kk = brev(register slot)
            // (plain stores: the column pass finds the last frames in L2).  Tiled output: x = lane + 32 kk lies in column tile
            // x / w = lane / w + kk (32 / w), so the stride between a lane's stores is 32 ny elements for every w
            const int w = a.tile_w;
            float2* out0 = a.out + (long long)f * npix + (w ? (long long)(lane / w) * a.ny * w + (long long)y * w + lane % w : (long long)y * NX + lane);
            const int es = w ? 32 * a.ny : 32;
#pragma unroll
            for (int p2 = 0; p2 < 32; ++p2) out0[brev<32>(p2) * es] = make_float2(o[p2].x, o[p2].y);
#pragma unroll
            for (int p2 = 0; p2 < 32; ++p2) out0[npix + brev<32>(p2) * es] = make_float2(o[p2].z, o[p2].w);
        } else {
            // (X[2 k], X[2 k + 1]) with k = lane + 32 kk: adjacent outputs, one 16-byte store
            float4* out0 = reinterpret_cast<float4*>(a.out + (long long)f * npix + (long long)y * NX) + lane;
#pragma unroll
            for (int p2 = 0; p2 < 32; ++p2) out0[32 * brev<32>(p2)] = o[p2];
        }
        tk0 = tk1;
        tk1 = __shfl_sync(0xffffffffu, tk2, 0);
    }
}

// ------------------------------------------------------------------------------------------------
// Mode 3 column pass for 2048-point columns, packed form: a CTA owns a tile of 8 columns (64-byte row segments); thread
// (j, c) holds elements n = j + 32 r and n + 1024 of column c, takes the radix-2 decimation-in-frequency step in registers
// (as k_rows2<2048>) and transforms the pair (y0, y1) with packed butterflies; the exchange goes through a padded CTA-wide
// buffer of 16-byte entries.  Outputs X(2k), X(2k+1) are two pixels: two accumulators per register slot.  Work units =
// (column tile, quarter of the frames), one CTA per SM; the quarters' partial images are added by k_sum_partial_images.
// Replaces the scalar three-pass kernel (4-column tiles, 32-byte segments, two exchanges) at N = 2048.
// ------------------------------------------------------------------------------------------------
struct C2Args {
    const float2* G;          // row-pass output [T][2048][nx]
    const float2* tw;         // [32][32] inter-pass twiddles of the 1024-point transform
    const float2* tw2048;     // exp(-2 pi i n / 2048), n < 1024
    float* out;               // ENERGY: [nsplit][2048][nx] partial images
    float2* H;                // !ENERGY: the hologram stack [T][2048][nx]
    int nx, T, nsplit;
};
constexpr int C2_B = 8;
constexpr int C2_SMEM = (F2N + F2N / 32) * C2_B * 16 + F2N * 8;

template <bool ENERGY>
__global__ void __launch_bounds__(256, 1) k_cols2048(const C2Args a) {
    extern __shared__ __align__(16) unsigned char smc_[];
    float4* ex = reinterpret_cast<float4*>(smc_);
    float2* tw_s = reinterpret_cast<float2*>(smc_ + (F2N + F2N / 32) * C2_B * 16);
    const int tid = threadIdx.x, j = tid / C2_B, c = tid % C2_B;
    for (int i = tid; i < F2N; i += 256) tw_s[i] = a.tw[i];
    auto sidx = [&](int i) -> int { return (i + i / 32) * C2_B + c; };
    const long long npix = 2048ll * a.nx;
    const int ntiles = a.nx / C2_B;
    const int per = (a.T + a.nsplit - 1) / a.nsplit;
    for (int unit = blockIdx.x; unit < ntiles * a.nsplit; unit += gridDim.x) {
        const int split = unit / ntiles, tile = unit - split * ntiles;       // split-major: concurrent CTAs walk adjacent tiles of the same frames
        const int t0 = split * per, t1 = t0 + per < a.T ? t0 + per : a.T;
        const float2* src0 = a.G + (long long)j * a.nx + (long long)tile * C2_B + c;
        float2 acc[ENERGY ? 32 : 1];
        if constexpr (ENERGY) {
#pragma unroll
            for (int r = 0; r < 32; ++r) acc[r] = make_float2(0.f, 0.f);
        }
        for (int t = t0; t < t1; ++t) {
            const float2* sa = src0 + (long long)t * npix;
            cpk v[32];
#pragma unroll
            for (int r = 0; r < 32; ++r) {
                const float2 xa = __ldcs(sa + (long long)(32 * r) * a.nx);
                const float2 xb = __ldcs(sa + (long long)(32 * r + 1024) * a.nx);
                v[r].re = make_float2(xa.x, xb.x); v[r].im = make_float2(xa.y, xb.y);       // (x(n), x(n + 1024)) for now
            }
#pragma unroll
            for (int r = 0; r < 32; ++r) {                     // y0 = x(n) + x(n + 1024), y1 = (x(n) - x(n + 1024)) W^n
                const float2 w = __ldg(a.tw2048 + j + 32 * r);
                const float sr = v[r].re.x + v[r].re.y, si = v[r].im.x + v[r].im.y;
                const float dr = v[r].re.x - v[r].re.y, di = v[r].im.x - v[r].im.y;
                v[r].re = make_float2(sr, fmaf(dr, w.x, -di * w.y));
                v[r].im = make_float2(si, fmaf(dr, w.y, di * w.x));
            }
            P2S<0, 5>::run(v);
            __syncthreads();                                   // the previous frame's exchange reads are over
#pragma unroll
            for (int r = 0; r < 32; ++r) { const cpk e = v[brev<32>(r)]; ex[sidx(j * 32 + r)] = make_float4(e.re.x, e.re.y, e.im.x, e.im.y); }
            __syncthreads();
#pragma unroll
            for (int r = 0; r < 32; ++r) { const float4 e = ex[sidx(j + 32 * r)]; v[r].re = make_float2(e.x, e.y); v[r].im = make_float2(e.z, e.w); }
#pragma unroll
            for (int r = 1; r < 32; ++r) {
                const float2 w = tw_s[r * 32 + j];
                const float2 re = pfma(w.x, v[r].re, pneg(__fmul2_rn(make_float2(w.y, w.y), v[r].im)));
                const float2 im = pfma(w.x, v[r].im, __fmul2_rn(make_float2(w.y, w.y), v[r].re));
                v[r].re = re; v[r].im = im;
            }
            P2S<0, 5>::run(v);
            if constexpr (ENERGY) {
#pragma unroll
                for (int r = 0; r < 32; ++r) {                 // k = j + 32 r: rows 2 k (first of the pair) and 2 k + 1
                    const cpk x = v[brev<32>(r)];
                    acc[r] = __ffma2_rn(x.re, x.re, __ffma2_rn(x.im, x.im, acc[r]));
                }
            } else {
                float2* hp = a.H + (long long)t * npix + (long long)(2 * j) * a.nx + (long long)tile * C2_B + c;
#pragma unroll
                for (int r = 0; r < 32; ++r) {
                    const cpk x = v[brev<32>(r)];
                    __stcs(hp + (long long)(64 * r) * a.nx, make_float2(x.re.x, x.im.x));
                    __stcs(hp + (long long)(64 * r + 1) * a.nx, make_float2(x.re.y, x.im.y));
                }
            }
        }
        if constexpr (ENERGY) {
            float* op = a.out + (long long)split * npix + (long long)(2 * j) * a.nx + (long long)tile * C2_B + c;
#pragma unroll
            for (int r = 0; r < 32; ++r) { op[(long long)(64 * r) * a.nx] = acc[r].x; op[(long long)(64 * r + 1) * a.nx] = acc[r].y; }
        }
    }
}

}  // namespace


// mode 3 row pass in the packed form: rows of 1024 points (even T: frame pairs) or of 2048 points (even / odd halves)
bool holo_rows2_supported(const holo_ctx* c) { return (c->nx == 1024 && (c->T % 2) == 0) || c->nx == 2048; }

int holo_launch_rows2(holo_ctx* c, const uint16_t* frames, float2* out, int ndefl, cudaStream_t st, int nframes, int tile_w) {
    R2Args a{};
    a.tile_w = c->nx == 1024 ? tile_w : 0;
    a.nframes = nframes > 0 ? nframes : c->T;
    a.frames = frames; a.sum = c->sum; a.qxs = c->qxs; a.qy = c->qy; a.tw = c->px.tw1;
    a.tw2048 = c->nx == 2048 ? c->px.tw2 + 1024 : nullptr;       // row r = 1 of the pass-2 table [2][1024]: exp(-2 pi i b / 2048)
    a.defl_img = c->defl_img; a.defl_coef = c->defl_coef; a.out = out; a.ticket = c->counters + 1001;
    a.T = c->T; a.ndefl = ndefl; a.ny = c->ny;
    int rc;
    HoloProf prof(c, HOLO_K_FFT_ROWS, st);
    if (c->nx == 1024) {
        if ((rc = holo_ensure_smem_attr((const void*)k_rows2<1024>, c->device, r2_smem<1024>()))) return rc;
        HOLO_CUDA_OK(holo_launch_pdl(k_rows2<1024>, dim3(c->num_sms - c->fresnel_sm_reserve), dim3(R2_WARPS * 32), r2_smem<1024>(), st, a));
    } else {
        if ((rc = holo_ensure_smem_attr((const void*)k_rows2<2048>, c->device, r2_smem<2048>()))) return rc;
        HOLO_CUDA_OK(holo_launch_pdl(k_rows2<2048>, dim3(c->num_sms - c->fresnel_sm_reserve), dim3(R2_WARPS * 32), r2_smem<2048>(), st, a));
    }
    HOLO_CUDA_OK(cudaGetLastError());
    return HOLO_OK;
}

// mode 3 column-energy pass in the packed form: columns of 2048 points.  `out` = image (nsplit = 1) or the partial images
bool holo_cols2048_supported(const holo_ctx* c) { return c->ny == 2048 && c->nx % C2_B == 0; }

int holo_launch_cols2048(holo_ctx* c, const float2* G, float* out, int nframes, int nsplit, cudaStream_t st) {
    C2Args a{};
    a.G = G; a.tw = c->py.tw1; a.tw2048 = c->py.tw2 + 1024; a.out = out; a.nx = c->nx; a.T = nframes; a.nsplit = nsplit;
    int rc;
    if ((rc = holo_ensure_smem_attr((const void*)k_cols2048<true>, c->device, C2_SMEM))) return rc;
    const int units = (c->nx / C2_B) * nsplit;
    HoloProf prof(c, HOLO_K_FFT_COLS, st);
    k_cols2048<true><<<units < c->num_sms ? units : c->num_sms, 256, C2_SMEM, st>>>(a);
    HOLO_CUDA_OK(cudaGetLastError());
    return HOLO_OK;
}

// the same column pass with the hologram stack as output (unfused Fresnel stage at 2048 x 2048)
int holo_launch_cols2048_store(holo_ctx* c, const float2* G, float2* H, int nframes, cudaStream_t st) {
    C2Args a{};
    a.G = G; a.tw = c->py.tw1; a.tw2048 = c->py.tw2 + 1024; a.H = H; a.nx = c->nx; a.T = nframes; a.nsplit = nframes >= 4 ? 4 : 1;
    int rc;
    if ((rc = holo_ensure_smem_attr((const void*)k_cols2048<false>, c->device, C2_SMEM))) return rc;
    const int units = (c->nx / C2_B) * a.nsplit;
    HoloProf prof(c, HOLO_K_FFT_COLS, st);
    const int sms = c->num_sms - c->fresnel_sm_reserve;    // (mode 2: one SM for the side-stream eigensolver)
    k_cols2048<false><<<units < sms ? units : sms, 256, C2_SMEM, st>>>(a);
    HOLO_CUDA_OK(cudaGetLastError());
    return HOLO_OK;
}
