// fft_reg.cuh -- register-level FFT building blocks shared by the Fresnel kernels (fresnel.cu, fresnel2.cu):
// compile-time twiddles, the radix-2 DIT butterfly network on scalar complex values, L2 cache-policy loads / stores and
// the release / acquire primitives of the persistent kernels.  Product code (CUDA, sm_100a); nothing here is shared
// with oracle/.
#pragma once
#include "holo_internal.cuh"

// ------------------------------------------------------------------------------------------------
// register FFT, radix-2 decimation in time, natural-order input, fully unrolled; the result is in
// bit-reversed order.  Stage s (s = 0 .. log2 R - 1) works in place on pairs at distance R/2^(s+1);
// the pairs of group g share the twiddle W_{2^(s+1)}^{rev_s(g)}.  A butterfly with a non-trivial
// twiddle costs 6 FMA-class instructions (tangent form: w b = wr (b_r - c b_i, b_i + c b_r), c = wi/wr,
// or the cotangent form when |wi| > |wr|) instead of 4 adds + 4 for the complex product.
// ------------------------------------------------------------------------------------------------
__host__ __device__ constexpr double cos32d(int k) {   // cos(2 pi k / 32), 0 <= k <= 16
    return k == 0 ? 1.0 : k == 1 ? 0.98078528040323044913 : k == 2 ? 0.92387953251128675613
         : k == 3 ? 0.83146961230254523708 : k == 4 ? 0.70710678118654752440 : k == 5 ? 0.55557023301960222474
         : k == 6 ? 0.38268343236508977173 : k == 7 ? 0.19509032201612826785 : k == 8 ? 0.0
         : -cos32d(16 - k);
}
__host__ __device__ constexpr double sin32d(int k) {   // sin(2 pi k / 32), 0 <= k <= 16
    return k <= 8 ? cos32d(8 - k) : cos32d(k - 8);
}
template <int R> __host__ __device__ constexpr int brev(int r) {
    int o = 0;
    for (int b = 1; b < R; b <<= 1) { o = (o << 1) | (r & 1); r >>= 1; }
    return o;
}

// (a, b) <- (a + w b, a - w b),  w = exp(-2 pi i E32 / 32), 0 <= E32 < 16
template <int E32> __host__ __device__ __forceinline__ void bfly_dit(float2& a, float2& b) {
    if constexpr (E32 == 0) {
        const float2 t = b;
        b = make_float2(a.x - t.x, a.y - t.y);
        a = make_float2(a.x + t.x, a.y + t.y);
    } else if constexpr (E32 == 8) {                      // w = -i: w b = (b_i, -b_r)
        const float2 t = b;
        b = make_float2(a.x - t.y, a.y + t.x);
        a = make_float2(a.x + t.y, a.y - t.x);
    } else {
        constexpr double wr = cos32d(E32), wi = -sin32d(E32);
        constexpr bool tanform = (wr < 0 ? -wr : wr) >= (wi < 0 ? -wi : wi);
        float tr, ti, sc;
        if constexpr (E32 == 4) { tr = b.x + b.y; ti = b.y - b.x; sc = (float)wr; }            // c = wi/wr = -1
        else if constexpr (E32 == 12) { tr = b.x - b.y; ti = b.y + b.x; sc = (float)wr; }      // c = +1
        else if constexpr (tanform) {
            constexpr float c = (float)(wi / wr);
            tr = fmaf(-c, b.y, b.x); ti = fmaf(c, b.x, b.y); sc = (float)wr;
        } else {
            constexpr float c = (float)(wr / wi);
            tr = fmaf(c, b.x, -b.y); ti = fmaf(c, b.y, b.x); sc = (float)wi;
        }
        b = make_float2(fmaf(-sc, tr, a.x), fmaf(-sc, ti, a.y));
        a = make_float2(fmaf(sc, tr, a.x), fmaf(sc, ti, a.y));
    }
}

template <int R, int S, int G, int M> struct DitM {      // pair M of group G in stage S
    static __host__ __device__ __forceinline__ void run(float2* v) {
        constexpr int span = R >> (S + 1);
        constexpr int e32 = brev<(1 << S)>(G) * (16 >> S);           // W_{2^(S+1)}^{rev_S(G)} as a 32nd root
        bfly_dit<e32>(v[2 * span * G + M], v[2 * span * G + M + span]);
        if constexpr (M + 1 < span) DitM<R, S, G, M + 1>::run(v);
    }
};
template <int R, int S, int G> struct DitG {
    static __host__ __device__ __forceinline__ void run(float2* v) {
        DitM<R, S, G, 0>::run(v);
        if constexpr (G + 1 < (1 << S)) DitG<R, S, G + 1>::run(v);
    }
};
template <int R, int S> struct DitS {
    static __host__ __device__ __forceinline__ void run(float2* v) {
        DitG<R, S, 0>::run(v);
        if constexpr ((2 << S) < R) DitS<R, S + 1>::run(v);
    }
};
// in-place DFT of size R (power of two <= 32) on registers v[0..R); X[r] = v[brev<R>(r)] afterwards
template <int R> __host__ __device__ __forceinline__ void fft_reg(float2* v) {
    if constexpr (R > 1) DitS<R, 0>::run(v);
}

__device__ __forceinline__ float2 cmul(float2 a, float2 b) {
    return make_float2(fmaf(-a.y, b.y, a.x * b.x), fmaf(a.y, b.x, a.x * b.y));
}

// L2 residency hints (createpolicy + ld/st .L2::cache_hint): the uint16 stack (64 MB at 1024^2 x 32) is kept
// in L2 between the sum kernel and the row pass, the row->column ring is kept until it is overwritten,
// and the hologram stores stream through (they are next read after 256 MB more have been written).
__device__ __forceinline__ uint64_t l2_evict_first() { uint64_t p; asm("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p)); return p; }
__device__ __forceinline__ uint64_t l2_evict_last() { uint64_t p; asm("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(p)); return p; }
__device__ __forceinline__ float2 ldcg_hint(const float2* p, uint64_t pol) {
    float2 v;
    asm volatile("ld.global.cg.L2::cache_hint.v2.f32 {%0,%1}, [%2], %3;" : "=f"(v.x), "=f"(v.y) : "l"(p), "l"(pol) : "memory");
    return v;
}
__device__ __forceinline__ void st_hint(float2* p, float2 v, uint64_t pol) {
    asm volatile("st.global.L2::cache_hint.v2.f32 [%0], {%1,%2}, %3;" ::"l"(p), "f"(v.x), "f"(v.y), "l"(pol) : "memory");
}
__device__ __forceinline__ int ldnc_u16_hint(const uint16_t* p, uint64_t pol) {
    unsigned short u;
    asm volatile("ld.global.nc.L2::cache_hint.u16 %0, [%1], %2;" : "=h"(u) : "l"(p), "l"(pol));
    return (int)u;
}
__device__ __forceinline__ uint4 ldnc_v4_hint(const uint4* p, uint64_t pol) {
    uint4 w;
    asm volatile("ld.global.nc.L2::cache_hint.v4.u32 {%0,%1,%2,%3}, [%4], %5;" : "=r"(w.x), "=r"(w.y), "=r"(w.z), "=r"(w.w) : "l"(p), "l"(pol));
    return w;
}

// ---- inter-CTA release / acquire on global counters (persistent kernels)
__device__ __forceinline__ unsigned int ld_acquire(const unsigned int* p) {
    unsigned int v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void red_release_add(unsigned int* p, unsigned int v) {
    asm volatile("red.release.gpu.global.add.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}

