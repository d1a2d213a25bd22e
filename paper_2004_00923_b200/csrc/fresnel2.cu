// fresnel2.cu -- A1 (mean-subtract + chirp prologue) and A2 (2-D FFT) for square frames of 1024 x 1024 pixels:
//   H_t = FFT2D[(I_t - mean_t I) * exp(+i pi (x^2+y^2)/(lambda z))]      (Eq. 1; R2-R6)
// Round-2 design: ONE persistent launch for all frames, like k_fresnel, but
//   * TWO sequences per thread in structure-of-arrays register pairs (re_a, re_b), (im_a, im_b): every butterfly of
//     the radix-32 networks is a packed FADD2 / FFMA2 on both sequences (same twiddle), i.e. half the FP32 issue
//     slots of the scalar form.  Row tiles pair the SAME row of two consecutive frames (one load of the frame sum S
//     and of the chirp serves both); column tiles pair two adjacent columns of one frame.
//   * 32 elements of each sequence per thread, so ONE WARP owns a pair of 1024-point sequences: pass 0 (radix 32),
//     one exchange through a warp-private, XOR-skewed shared-memory region (16-byte accesses, conflict free), pass 1
//     (radix 32).  Only __syncwarp inside a tile -- no CTA-wide barrier anywhere in the steady state.
//   * column tiles ([1024 rows x 8 columns], 64 KB) are brought in and written out by the TMA unit
//     (cp.async.bulk.tensor, 64-byte rows, SWIZZLE_64B) straight into / out of the buffer the four warps of a group
//     transform IN PLACE.  Three autonomous groups of four warps per SM, each with its own buffer and its own
//     scheduler lane (tickets drawn one tile ahead, dependency wait, TMA issue; mbarrier full / done pairs): while
//     one group waits for its tile to land the other two compute.  The compute warps never touch the LSU with
//     uncoalesced addresses.
//   * the first radix-2 stage of a column tile reads the array-of-structures complex values TMA delivered and writes
//     SoA pairs, the last stage of every tile writes AoS again: the layout change costs no move instructions.
// Ticket order, ring of R frames between the passes and the release / acquire counters follow k_fresnel, in units of
// frame pairs.
#include "holo_internal.cuh"
#include "fft_reg.cuh"
#include "tma.cuh"
#include <vector>

#ifdef F2_TIMING
__device__ __forceinline__ unsigned long long f2_gt() { unsigned long long t; asm volatile("mov.u64 %0, %globaltimer;" : "=l"(t)); return t; }
#define F2_TR(slot) do { if (lane == 5 && wg == 1 && a.trace) a.trace[(size_t)cur_tk * 8 + (slot)] = f2_gt(); } while (0)
#define F2_T(i) do { const unsigned int _c = (unsigned int)clock(); f2_tacc[i] += _c - f2_tlast; f2_tlast = _c; } while (0)
#else
#define F2_T(i) do {} while (0)
#define F2_TR(slot) do {} while (0)
#endif

namespace {

constexpr int F2N = 1024;                 // sequence length (rows and columns)
constexpr int F2_TILE = 65536;            // bytes of one tile buffer: 8 sequences x 1024 x 8 B
constexpr int F2_GROUPS = 3;              // autonomous groups of 4 warps, one tile buffer each
constexpr int F2_THREADS = 4 * F2_GROUPS * 32;
constexpr int F2_RT = F2N / 8;            // row tiles per frame (8 rows each: 4 warps x 2 adjacent rows)
constexpr int F2_CT = F2N / 8;            // column tiles per frame (8 columns each)
constexpr int F2_SMEM = 1024 + F2_GROUPS * F2_TILE + 2 * F2N * 8 + 256;

struct F2Args {
    const uint16_t* frames;   // [nframes][N][N]
    const uint32_t* sum;      // S = sum_t I_t
    const float2* qxs;        // chirp along x, scaled by 1/T
    const float2* qy;         // chirp along y
    const float2* tw;         // [32][32] inter-pass twiddles exp(-2 pi i r k / 1024)
    float2* ring;             // [R][N][N] row -> column intermediate
    unsigned long long* trace; // F2_TIMING builds: [ticket][8] global-timer stamps of warp 1 of the group
    unsigned int* timing;     // F2_TIMING builds: [warp slot][16] accumulated cycles per phase
    unsigned int* counters;   // [0] ticket, [1 + f] rows_done (warps), [1 + T + f] cols_done (tiles landed)
    int nframes, T, R, L;     // frames to transform, stack length (d = T I - S), ring frames, lag in frames
};

struct F2Desc { int flags, rf, rw, cf, cw, ring_ok, tk, pad2; };   // row tile rw of frame rf and / or column tile cw of frame cf
enum { F2_ROW = 1, F2_COL = 2, F2_EXIT = 4 };

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
__device__ __forceinline__ void red_relaxed_add(unsigned int* p, unsigned int v) {
    asm volatile("red.relaxed.gpu.global.add.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
__device__ __forceinline__ void tma_2d_s2g_hint(const CUtensorMap* tm, int c0, int c1, uint32_t src_smem, uint64_t pol) {
    asm volatile("cp.async.bulk.tensor.2d.global.shared::cta.bulk_group.L2::cache_hint [%0, {%1, %2}], [%3], %4;"
                 ::"l"(tm), "r"(c0), "r"(c1), "r"(src_smem), "l"(pol) : "memory");
}
__device__ __forceinline__ void tma_2d_g2s_hint(void* dst_smem, const CUtensorMap* tm, int c0, int c1, uint64_t* bar, uint64_t pol) {
    asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1, {%2, %3}], [%4], %5;"
                 ::"r"(smem_u32(dst_smem)), "l"(tm), "r"(c0), "r"(c1), "r"(smem_u32(bar)), "l"(pol) : "memory");
}
__device__ __forceinline__ unsigned int ld_relaxed(const unsigned int* p) {
    unsigned int v;
    asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
// wait until *p >= need (polling without the L1 invalidation an acquire load carries), then acquire once
__device__ __forceinline__ void wait_counter(const unsigned int* p, unsigned int need) {
    while (ld_relaxed(p) < need) __nanosleep(100);
    asm volatile("fence.acq_rel.gpu;" ::: "memory");
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

// ---- row tile: rows r, r+1 of frame f (one warp) ---------------------------------------------------------------
// `before_exchange` / `after_exchange` bracket the warp's use of the shared buffer; `before_store` returns once the
// ring slot of the frame may be overwritten.
template <class Before, class After, class Store>
__device__ __forceinline__ void row_tile(const F2Args& a, int f, int r, uint32_t buf, int wg, int lane,
                                         const float2* tw_s, const float2* qx_s, Before before_exchange, After after_exchange,
                                         Store before_store, unsigned int* f2_tacc, unsigned int& f2_tlast) {
    const long long npix = (long long)F2N * F2N;
    const uint16_t* I0 = a.frames + (long long)f * npix + (long long)r * F2N + lane;
    const uint32_t* Sp = a.sum + (long long)r * F2N + lane;
    const uint64_t pol_in = l2_evict_first();
    const float2 qy0 = __ldg(a.qy + r), qy1 = __ldg(a.qy + r + 1);
    const float Tf = (float)a.T;
    const XAddr xa = make_xaddr(buf, wg, lane);
    cpk v[32];
    // pass 0 inputs: x = lane + 32 m.  d = T I - S exactly: uint -> float through the 2^23 trick (values < 2^23),
    // then one FMA; the 1/T lives in the qx table.  All loads of the tile are issued before the first use.
    {
        unsigned int u0[32], u1[32], s0[32], s1[32];
#pragma unroll
        for (int m = 0; m < 32; ++m) {
            u0[m] = (unsigned int)ldnc_u16_hint(I0 + 32 * m, pol_in);
            u1[m] = (unsigned int)ldnc_u16_hint(I0 + F2N + 32 * m, pol_in);
            s0[m] = __ldg(Sp + 32 * m);
            s1[m] = __ldg(Sp + F2N + 32 * m);
        }
#pragma unroll
        for (int m = 0; m < 32; ++m) {
            const float2 magic = make_float2(-8388608.f, -8388608.f);
            const float2 fi = __fadd2_rn(make_float2(__uint_as_float(0x4B000000u | u0[m]), __uint_as_float(0x4B000000u | u1[m])), magic);
            const float2 fs = __fadd2_rn(make_float2(__uint_as_float(0x4B000000u | s0[m]), __uint_as_float(0x4B000000u | s1[m])), magic);
            const float2 d = __ffma2_rn(make_float2(Tf, Tf), fi, pneg(fs));
            const float2 qx = qx_s[lane + 32 * m];
            const float2 q0 = cmul(qx, qy0), q1 = cmul(qx, qy1);
            v[m].re = __fmul2_rn(d, make_float2(q0.x, q1.x));
            v[m].im = __fmul2_rn(d, make_float2(q0.y, q1.y));
        }
    }
    F2_T(1);
    P2S<0, 5>::run(v);
    F2_T(2);
    before_exchange();
    F2_T(3);
    exchange_write(xa, v);
    __syncwarp();
    exchange_read_twiddle(xa, v, tw_s, lane);
    __syncwarp();                                   // every lane has read: the warp no longer needs the buffer
    F2_T(4);
    after_exchange();
    F2_T(5);
    P2S<0, 4>::run(v);
    float4 o[32];
    P2Last<0>::run(v, o);
    F2_T(6);
    before_store();
    F2_T(7);
    // X[lane + 32 kk] of row r in (o.x, o.y), of row r+1 in (o.z, o.w); kk = brev(register slot)
    const uint64_t pol_out = l2_evict_last();
    float2* out0 = a.ring + (long long)(f % a.R) * npix + (long long)r * F2N + lane;
#pragma unroll
    for (int p = 0; p < 32; ++p) st_hint(out0 + 32 * brev<32>(p), make_float2(o[p].x, o[p].y), pol_out);
#pragma unroll
    for (int p = 0; p < 32; ++p) st_hint(out0 + F2N + 32 * brev<32>(p), make_float2(o[p].z, o[p].w), pol_out);
}

// ---- column tile: columns (c, c+1) of one frame, delivered by TMA into the warp's chunk of the buffer ----------
template <class Mid>
__device__ __forceinline__ void col_tile(uint32_t buf, int wg, int lane, const float2* tw_s, unsigned int* landed, Mid mid,
                                         unsigned int* f2_tacc, unsigned int& f2_tlast) {
    const XAddr xa = make_xaddr(buf, wg, lane);
    cpk v[32];
    {
        float4 x[32];                                // AoS (re_c, im_c, re_c+1, im_c+1) of rows lane + 32 m
#pragma unroll
        for (int m = 0; m < 32; ++m) x[m] = lds128(xa.nat + 2048u * m);
        __syncwarp();                                // every lane has its inputs before the exchange overwrites the rows
        // the ring rows of this tile have left global memory: the frame's ring slot may be reused once all its tiles say so
        if (wg == 0 && lane == 0) red_relaxed_add(landed, 1u);
        // stage 0 of the DIT network (pairs (m, m + 16), w = 1) reads AoS, writes SoA
#pragma unroll
        for (int m = 0; m < 16; ++m) {
            const float4 p = x[m], q = x[m + 16];
            v[m].re = make_float2(p.x + q.x, p.z + q.z); v[m].im = make_float2(p.y + q.y, p.w + q.w);
            v[m + 16].re = make_float2(p.x - q.x, p.z - q.z); v[m + 16].im = make_float2(p.y - q.y, p.w - q.w);
        }
    }
    P2S<1, 5>::run(v);
    F2_T(10);
    exchange_write(xa, v);
    __syncwarp();
    exchange_read_twiddle(xa, v, tw_s, lane);
    __syncwarp();
    mid();
    F2_T(11);
    P2S<0, 4>::run(v);
    float4 o[32];
    P2Last<0>::run(v, o);
    F2_T(12);
    // H[lane + 32 kk][c, c+1] -> row lane + 32 kk of the buffer, in the layout the TMA store expects
#pragma unroll
    for (int p = 0; p < 32; ++p) sts128(xa.nat + 2048u * brev<32>(p), o[p]);
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}

// A ticket is a SUPER-TILE: row tile i of frame f together with column tile i of frame f - L (whose row pass ended
// L blocks of 128 tickets ago).  Order: rows(0..L-1) alone, [rows(f) + cols(f - L)] for f = L..n-1, cols(n-L..n-1)
// alone.  Every dependency of a ticket has a smaller ticket.
__device__ __forceinline__ void f2_decode(const F2Args& a, unsigned int tk, F2Desc& d) {
    const int b = (int)(tk / F2_RT), i = (int)(tk % F2_RT);
    d.flags = 0; d.rf = d.rw = d.cf = d.cw = 0; d.ring_ok = 1; d.tk = (int)tk; d.pad2 = 0;
    if (b < a.nframes) { d.flags |= F2_ROW; d.rf = b; d.rw = i; }
    if (b >= a.L) { d.flags |= F2_COL; d.cf = b - a.L; d.cw = i; }
}

// One persistent CTA per SM, three autonomous groups of four warps, one 64 KB buffer per group.  Lane 0 of a group's
// first warp (the leader) is its scheduler: it holds the next ticket (drawn one super-tile ahead, so the atomic's round
// trip is hidden) and waits for the dependencies.  Within a super-tile the buffer is used twice: as the exchange area of
// the row tile, then -- as soon as the four warps have read their exchange back, i.e. while they still compute pass 1
// and store their rows -- as the landing zone of the column tile's TMA load; the column tile is transformed in place
// and leaves through a TMA store whose drain hides behind the global loads of the next row tile.
// mbarriers per group: full (ticket published), xdone (4 warps: exchange read), land (column tile landed),
// cdone (4 warps: column results in the buffer), drained (the store has read the buffer).
__global__ void __launch_bounds__(F2_THREADS, 1)
k_fresnel2(const __grid_constant__ CUtensorMap tmRing, const __grid_constant__ CUtensorMap tmH, const F2Args a) {
    extern __shared__ unsigned char smraw_[];
    // 1024-byte aligned tile buffers (the TMA swizzle pattern is a function of the shared-memory address)
    const uint32_t s0 = smem_u32(smraw_);
    const uint32_t pad = (1024u - (s0 & 1023u)) & 1023u;
    unsigned char* base = smraw_ + pad;
    const uint32_t bufs = s0 + pad;
    float2* tw_s = reinterpret_cast<float2*>(base + F2_GROUPS * F2_TILE);
    float2* qx_s = tw_s + F2N;
    uint64_t* bars = reinterpret_cast<uint64_t*>(qx_s + F2N);          // [group][5]
    F2Desc* desc = reinterpret_cast<F2Desc*>(bars + 5 * F2_GROUPS);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;

    for (int i = tid; i < F2N; i += F2_THREADS) { tw_s[i] = a.tw[i]; qx_s[i] = a.qxs[i]; }
    if (tid == 0) {
        for (int s = 0; s < F2_GROUPS; ++s) {
            mbar_init(bars + 5 * s + 0, 1); mbar_init(bars + 5 * s + 1, 4); mbar_init(bars + 5 * s + 2, 1);
            mbar_init(bars + 5 * s + 3, 4); mbar_init(bars + 5 * s + 4, 1);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    const unsigned int total = (unsigned int)(a.nframes + a.L) * F2_RT;
    const int g = warp >> 2, wg = warp & 3;
    const bool leader = wg == 0 && lane == 0;
    const uint32_t buf = bufs + (uint32_t)g * F2_TILE;
    unsigned char* bufp = base + (size_t)g * F2_TILE;
    uint64_t* full = bars + 5 * g; uint64_t* xdone = full + 1; uint64_t* land = full + 2; uint64_t* cdone = full + 3; uint64_t* drained = full + 4;
    uint32_t ph_full = 0, ph_x = 0, ph_land = 0, ph_c = 0, ph_dr = 0;
    bool store_pending = false;                  // the previous super-tile's TMA store may still be reading the buffer
    unsigned int* pending_rel = nullptr;         // rows_done counter of a row tile whose stores have not been announced yet
    unsigned int nt = 0u;                        // leader: the next ticket
    if (leader) nt = atomicAdd(a.counters, 1u);
    unsigned int f2_tacc[16] = {0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0};
    unsigned int f2_tlast = (unsigned int)clock();

    auto issue_col_load = [&](const F2Desc& d) {                       // leader only; the buffer is free
        wait_counter(a.counters + 1 + d.cf, 4u * F2_RT);                // the row pass of the frame is complete
        asm volatile("fence.proxy.async;" ::: "memory");                // ring rows were written through the generic proxy
        mbar_arrive_expect_tx(land, (uint32_t)F2_TILE);
        const uint64_t pol = l2_evict_last();
#pragma unroll
        for (int q = 0; q < 4; ++q)
            tma_2d_g2s_hint(bufp + (size_t)q * 16384, &tmRing, 16 * d.cw, (d.cf % a.R) * F2N + 256 * q, land, pol);
    };

#pragma unroll 1
    for (;;) {
        if (leader) {
            F2Desc d;
            const unsigned int tk = nt;
            if (tk < total) f2_decode(a, tk, d);
            if (tk >= total) {
                d.flags = F2_EXIT;
                desc[g] = d;
                mbar_arrive(full);
            } else {
                // has the ring slot of the row tile's frame been read by every column tile of frame rf - R?  Looked at now,
                // waited for (if need be) only just before the rows are stored
                if ((d.flags & F2_ROW) && d.rf >= a.R) d.ring_ok = ld_relaxed(a.counters + 1 + a.T + d.rf - a.R) >= (unsigned int)F2_CT;
                desc[g] = d;
                mbar_arrive(full);
                if (!(d.flags & F2_ROW)) {                               // column tile alone (tail of the launch)
                    if (store_pending) asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
                    issue_col_load(d);
                }
            }
        }
        mbar_wait(full, ph_full); ph_full ^= 1u;
        F2_T(0);
        const F2Desc d = desc[g];
        if (d.flags & F2_EXIT) break;
        const int cur_tk = d.tk; (void)cur_tk;
        F2_TR(0);
        if (d.flags & F2_ROW) {
            auto before_exchange = [&]() {
                F2_TR(1);
                if (store_pending) {                                      // uniform over the group
                    if (leader) { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); mbar_arrive(drained); }
                    mbar_wait(drained, ph_dr); ph_dr ^= 1u;
                }
            };
            auto after_exchange = [&]() {                                 // this warp no longer needs the buffer
                F2_TR(2);
                if (lane == 0) mbar_arrive(xdone);
                if (leader && (d.flags & F2_COL)) { mbar_wait(xdone, ph_x); issue_col_load(d); }
                if (leader && !(d.flags & F2_COL)) nt = atomicAdd(a.counters, 1u);     // row tile alone: draw the next ticket here
                ph_x ^= 1u;
            };
            auto before_store = [&]() {
                F2_TR(3);
                if (!d.ring_ok) {                                         // rare: uniform over the group
                    if (lane == 0) wait_counter(a.counters + 1 + a.T + d.rf - a.R, (unsigned int)F2_CT);
                    __syncwarp();
                }
                F2_TR(4);
            };
            row_tile(a, d.rf, 8 * d.rw + 2 * wg, buf, wg, lane, tw_s, qx_s, before_exchange, after_exchange, before_store, f2_tacc, f2_tlast);
            F2_T(8);
            // the rows are announced (release) only in the middle of the column tile that follows, when the stores have long
            // drained: a release right here would stall the warp for the whole store latency (measured 4 us per tile)
            __syncwarp();
            pending_rel = a.counters + 1 + d.rf;
            if (!(d.flags & F2_COL)) { if (lane == 0) red_release_add(pending_rel, 1u); pending_rel = nullptr; }
            F2_T(9);
            F2_TR(5);
        }
        store_pending = false;
        if (d.flags & F2_COL) {
            // the next ticket is drawn as late as its round trip allows: tickets drawn a whole super-tile ahead would double the
            // window of tickets in flight, and with it the ring depth the dependencies need
            if (leader) nt = atomicAdd(a.counters, 1u);
            mbar_wait(land, ph_land); ph_land ^= 1u;
            F2_T(13);
            F2_TR(6);
            auto col_mid = [&]() { if (pending_rel) { if (lane == 0) red_release_add(pending_rel, 1u); pending_rel = nullptr; } };
            col_tile(buf, wg, lane, tw_s, a.counters + 1 + a.T + d.cf, col_mid, f2_tacc, f2_tlast);
            F2_T(14);
            F2_TR(7);
            __syncwarp();
            if (lane == 0) mbar_arrive(cdone);
            if (leader) {
                mbar_wait(cdone, ph_c);
                const uint64_t pol = l2_evict_first();
#pragma unroll
                for (int q = 0; q < 4; ++q) tma_2d_s2g_hint(&tmH, 16 * d.cw, d.cf * F2N + 256 * q, buf + (uint32_t)q * 16384u, pol);
                asm volatile("cp.async.bulk.commit_group;" ::: "memory");
            }
            ph_c ^= 1u;
            store_pending = true;
            F2_T(15);
        }
    }
#ifdef F2_TIMING
    if (a.timing) for (int i = 0; i < 16; ++i) a.timing[((size_t)blockIdx.x * (F2_THREADS / 32) + warp) * 32 * 16 + lane * 16 + i] = f2_tacc[i];
#endif
    if (leader) asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
}

// ------------------------------------------------------------------------------------------------
// Mode 3 row pass, packed form (1024-point rows): one warp transforms row y of TWO consecutive frames (f, f + 1) at once.
// The frame sum S, the deflation images e_k and the chirp of the row are loaded once for both, every butterfly is a
// packed FADD2 / FFMA2 on the pair, the exchange uses 16-byte accesses: about 60 % of the instructions and of the L1
// traffic of the scalar row kernel (k_fft), which ncu shows bound by instruction issue (58 %) and the L1 pipe (72 %).
// Warps are autonomous (row pairs drawn from a ticket, warp-private exchange slice, no CTA-wide step).
// ------------------------------------------------------------------------------------------------
struct R2Args {
    const uint16_t* frames;   // [T][N][N]
    const uint32_t* sum;      // S = sum_t I_t
    const float2* qxs;        // chirp along x, scaled by 1/T
    const float2* qy;
    const float2* tw;         // [32][32] inter-pass twiddles
    const float* defl_img;    // [ndefl][N][N]  eT_k
    const float* defl_coef;   // [T][ndefl]
    float2* out;              // [T][N][N] row-pass output
    unsigned int* ticket;     // zeroed by an earlier kernel of the stream
    int T, ndefl;
};

constexpr int R2_WARPS = 12;
constexpr int R2_SMEM = 1024 + (R2_WARPS / 4) * F2_TILE + 2 * F2N * 8;

__global__ void __launch_bounds__(R2_WARPS * 32, 1) k_rows2(const R2Args a) {
    extern __shared__ unsigned char smraw_[];
    const uint32_t s0 = smem_u32(smraw_);
    const uint32_t pad = (1024u - (s0 & 1023u)) & 1023u;
    unsigned char* base = smraw_ + pad;
    const uint32_t bufs = s0 + pad;
    float2* tw_s = reinterpret_cast<float2*>(base + (R2_WARPS / 4) * F2_TILE);
    float2* qx_s = tw_s + F2N;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    for (int i = tid; i < F2N; i += R2_WARPS * 32) { tw_s[i] = a.tw[i]; qx_s[i] = a.qxs[i]; }
    __syncthreads();
    const uint32_t buf = bufs + (uint32_t)(warp >> 2) * F2_TILE;
    const XAddr xa = make_xaddr(buf, warp & 3, lane);
    const long long npix = (long long)F2N * F2N;
    const unsigned int npairs = (unsigned int)(a.T / 2) * F2N;
    const float Tf = (float)a.T;
    // tickets are drawn two tasks ahead (the atomic's round trip is hidden) and the frame rows of the NEXT task are pulled
    // into L2 while the current one computes (ncu: 14 % of the warp time waited for the ticket, 30 % for the loads)
    unsigned int tk0 = 0u, tk1 = 0u;
    if (lane == 0) { tk0 = atomicAdd(a.ticket, 1u); tk1 = atomicAdd(a.ticket, 1u); }
    tk0 = __shfl_sync(0xffffffffu, tk0, 0); tk1 = __shfl_sync(0xffffffffu, tk1, 0);
    for (;;) {
        const unsigned int tk = tk0;
        if (tk >= npairs) break;
        unsigned int tk2 = 0u;
        if (lane == 0) tk2 = atomicAdd(a.ticket, 1u);
        if (tk1 < npairs) {
            const int f1 = 2 * (int)(tk1 / F2N), y1 = (int)(tk1 % F2N);
            const uint16_t* pf = a.frames + (long long)(f1 + (lane >> 4)) * npix + (long long)y1 * F2N + (lane & 15) * 64;
            asm volatile("prefetch.global.L2 [%0];" ::"l"(pf));
        }
        const int f = 2 * (int)(tk / F2N), y = (int)(tk % F2N);
        const uint16_t* Ia = a.frames + (long long)f * npix + (long long)y * F2N + lane;
        const uint32_t* Sp = a.sum + (long long)y * F2N + lane;
        const float2 qyv = __ldg(a.qy + y);
        cpk v[32];
        // d = T I - S exactly (integers below 2^23); the pair (frame f, frame f + 1) in the two halves of a packed value
#pragma unroll
        for (int m = 0; m < 32; ++m) {
            const float ia = (float)__ldg(Ia + 32 * m), ib = (float)__ldg(Ia + npix + 32 * m);
            const float sv = (float)__ldg(Sp + 32 * m);
            v[m].re = make_float2(fmaf(Tf, ia, -sv), fmaf(Tf, ib, -sv));
        }
        const float* ep = a.defl_img + (long long)y * F2N + lane;
        for (int kk = 0; kk < a.ndefl; ++kk) {
            const float2 cf = make_float2(-__ldg(a.defl_coef + f * a.ndefl + kk), -__ldg(a.defl_coef + (f + 1) * a.ndefl + kk));
            float e[32];
#pragma unroll
            for (int m = 0; m < 32; ++m) e[m] = __ldg(ep + 32 * m);
#pragma unroll
            for (int m = 0; m < 32; ++m) v[m].re = __ffma2_rn(make_float2(e[m], e[m]), cf, v[m].re);
            ep += npix;
        }
#pragma unroll
        for (int m = 0; m < 32; ++m) {
            const float2 q = cmul(qx_s[lane + 32 * m], qyv);
            const float2 d = v[m].re;
            v[m].re = __fmul2_rn(d, make_float2(q.x, q.x));
            v[m].im = __fmul2_rn(d, make_float2(q.y, q.y));
        }
        P2S<0, 5>::run(v);
        exchange_write(xa, v);
        __syncwarp();
        exchange_read_twiddle(xa, v, tw_s, lane);
        __syncwarp();
        P2S<0, 4>::run(v);
        float4 o[32];
        P2Last<0>::run(v, o);
        // X[lane + 32 kk] of frame f in (o.x, o.y), of frame f + 1 in (o.z, o.w); kk = brev(register slot)
        float2* out0 = a.out + (long long)f * npix + (long long)y * F2N + lane;
#pragma unroll
        for (int p2 = 0; p2 < 32; ++p2) __stcs(out0 + 32 * brev<32>(p2), make_float2(o[p2].x, o[p2].y));
#pragma unroll
        for (int p2 = 0; p2 < 32; ++p2) __stcs(out0 + npix + 32 * brev<32>(p2), make_float2(o[p2].z, o[p2].w));
        tk0 = tk1;
        tk1 = __shfl_sync(0xffffffffu, tk2, 0);
    }
}

int make_map_2d(CUtensorMap* tm, const void* base, unsigned long long dim0_floats, unsigned long long rows, unsigned long long row_bytes,
                unsigned int box0, unsigned int box1, CUtensorMapSwizzle swz) {
    static EncodeTiledFn encode = nullptr;
    if (!encode) {
        void* fn = nullptr;
        cudaDriverEntryPointQueryResult qres;
        HOLO_CUDA_OK(cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres));
        if (!fn || qres != cudaDriverEntryPointSuccess) { holo_set_error("cuTensorMapEncodeTiled not available"); return HOLO_ERR_CUDA; }
        encode = (EncodeTiledFn)fn;
    }
    const cuuint64_t gdim[2] = {(cuuint64_t)dim0_floats, (cuuint64_t)rows};
    const cuuint64_t gstr[1] = {(cuuint64_t)row_bytes};
    const cuuint32_t box[2] = {box0, box1};
    const cuuint32_t estr[2] = {1, 1};
    const CUresult r = encode(tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, const_cast<void*>(base), gdim, gstr, box, estr,
                              CU_TENSOR_MAP_INTERLEAVE_NONE, swz, CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) { holo_set_error("cuTensorMapEncodeTiled failed (%d)", (int)r); return HOLO_ERR_CUDA; }
    return HOLO_OK;
}

}  // namespace

bool holo_fresnel2_supported(const holo_ctx* c) {
    return c->nx == F2N && c->ny == F2N && c->scratch_frames >= 2;
}

// frames[0..nproc) -> H[0..nproc); c->sum holds S, c->counters are zero (k_frame_sum or a memset did that)
int holo_launch_fresnel2(holo_ctx* c, const uint16_t* frames, float2* H, cudaStream_t st, int nproc) {
    F2Args a{};
    a.frames = frames; a.sum = c->sum; a.qxs = c->qxs; a.qy = c->qy; a.tw = c->px.tw1;
    a.ring = c->scratch; a.counters = c->counters;
#ifdef F2_TIMING
    static unsigned int* tbuf = nullptr;
    static unsigned long long* trbuf = nullptr;
    if (!tbuf) { cudaMalloc(&tbuf, (size_t)148 * 12 * 32 * 16 * 4); cudaMalloc(&trbuf, (size_t)8192 * 8 * 8); }
    cudaMemsetAsync(trbuf, 0, (size_t)8192 * 8 * 8, st);
    a.timing = tbuf; a.trace = trbuf;
#endif
    a.nframes = nproc; a.T = c->T;
    a.R = c->scratch_frames;
    int L = c->tune[HOLO_TUNE_FFT_LAG] > 0 ? c->tune[HOLO_TUNE_FFT_LAG] : a.R / 2;
    if (L > a.R - 1) L = a.R - 1;                // rows(f) waits for cols(f - R), whose tickets must precede its own
    if (L > nproc) L = nproc;
    if (L < 1) L = 1;
    a.L = L;
    alignas(64) CUtensorMap tmRing, tmH;
    int rc;
    if ((rc = make_map_2d(&tmRing, c->scratch, 2ull * F2N, (unsigned long long)a.R * F2N, (unsigned long long)F2N * 8, 16, 256, CU_TENSOR_MAP_SWIZZLE_64B))) return rc;
    if ((rc = make_map_2d(&tmH, H, 2ull * F2N, (unsigned long long)nproc * F2N, (unsigned long long)F2N * 8, 16, 256, CU_TENSOR_MAP_SWIZZLE_64B))) return rc;
    if ((rc = holo_ensure_smem_attr((const void*)k_fresnel2, c->device, F2_SMEM))) return rc;
    const long long total = (long long)(nproc + L) * F2_RT;
    long long grid = c->num_sms;                          // one persistent CTA per SM (all co-resident)
    if (grid * F2_GROUPS > total) grid = (total + F2_GROUPS - 1) / F2_GROUPS;   // (a group without a ticket exits at once)
    HoloProf prof(c, HOLO_K_FFT_ROWS, st);
    k_fresnel2<<<(int)grid, F2_THREADS, F2_SMEM, st>>>(tmRing, tmH, a);
    HOLO_CUDA_OK(cudaGetLastError());
#ifdef F2_TIMING
    {
        cudaStreamSynchronize(st);
        static int calls = 0;
        if (++calls == 20) {
            std::vector<unsigned int> h((size_t)148 * 12 * 32 * 16);
            cudaMemcpy(h.data(), tbuf, h.size() * 4, cudaMemcpyDeviceToHost);
            double acc[2][16] = {};
            for (int w = 0; w < 148 * 12; ++w) for (int i = 0; i < 16; ++i) { acc[0][i] += h[((size_t)w * 32 + 0) * 16 + i]; acc[1][i] += h[((size_t)w * 32 + 5) * 16 + i]; }
            { std::vector<unsigned long long> tr((size_t)8192 * 8); cudaMemcpy(tr.data(), trbuf, tr.size() * 8, cudaMemcpyDeviceToHost);
              FILE* fp = fopen("gpurun_out/f2_trace.bin", "wb"); if (fp) { fwrite(tr.data(), 8, tr.size(), fp); fclose(fp); } }
            for (int l = 0; l < 2; ++l) { fprintf(stderr, "F2_TIMING lane %d (avg cycles per warp per launch):", l ? 5 : 0); double t = 0; for (int i = 0; i < 16; ++i) { fprintf(stderr, " [%d]%.0f", i, acc[l][i] / (148 * 12)); t += acc[l][i] / (148 * 12); } fprintf(stderr, " total %.0f\n", t); }
        }
    }
#endif
    return HOLO_OK;
}

// mode 3 row pass in the packed form: supported for 1024 x 1024 frames and even T
bool holo_rows2_supported(const holo_ctx* c) { return c->nx == F2N && c->ny == F2N && (c->T % 2) == 0; }

int holo_launch_rows2(holo_ctx* c, const uint16_t* frames, float2* out, int ndefl, cudaStream_t st) {
    R2Args a{};
    a.frames = frames; a.sum = c->sum; a.qxs = c->qxs; a.qy = c->qy; a.tw = c->px.tw1;
    a.defl_img = c->defl_img; a.defl_coef = c->defl_coef; a.out = out; a.ticket = c->counters + 1001;
    a.T = c->T; a.ndefl = ndefl;
    int rc;
    if ((rc = holo_ensure_smem_attr((const void*)k_rows2, c->device, R2_SMEM))) return rc;
    HoloProf prof(c, HOLO_K_FFT_ROWS, st);
    k_rows2<<<c->num_sms, R2_WARPS * 32, R2_SMEM, st>>>(a);
    HOLO_CUDA_OK(cudaGetLastError());
    return HOLO_OK;
}
