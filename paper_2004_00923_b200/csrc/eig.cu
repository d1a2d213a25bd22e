// eig.cu -- A4: C = V Lambda V^{t*}   (Eq. 5; R1 descending order, R8, R10, R11)
//
// Single-CTA two-sided complex Hermitian Jacobi in FP32, parallel (round-robin tournament) ordering:
// each of the Tp-1 steps of a sweep annihilates Tp/2 disjoint pivots at once.  A and V live in
// shared memory in SYSTOLIC (Brent-Luk) arrangement: the pivot pairs of every step are the
// positions (2b, 2b+1); after the rotations each row/column is written to the position it takes in
// the next step (a fixed permutation), so a thread's read and write addresses never change and
// the step body carries no index arithmetic -- the kernel is bound by the latency of one step
// (shared-memory round trip + rotation parameters + 2x2 update + one barrier), not by throughput.
// After convergence the eigenvalues are refined as FP64 Rayleigh quotients v_k^H C v_k of the
// ORIGINAL matrix, sorted descending, and every eigenvector is normalised and phase-fixed
// (largest-magnitude entry real positive, ties -> lowest index).
#include "holo_internal.cuh"

__device__ __forceinline__ float2 cmulf(float2 a, float2 b) {
    return make_float2(fmaf(-a.y, b.y, a.x * b.x), fmaf(a.y, b.x, a.x * b.y));
}
__device__ __forceinline__ float2 cmulcf(float2 a, float2 b) {      // a * conj(b)
    return make_float2(fmaf(a.y, b.y, a.x * b.x), fmaf(a.y, b.x, -a.x * b.y));
}
__device__ __forceinline__ float rsqrt_fast(float x) { float y; asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float rcp_fast(float x) { float y; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }

__device__ float block_sum(float v, float* red) {       // all threads must call; result broadcast
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = blockDim.x >> 5;
#pragma unroll
    for (int o = 16; o >= 1; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    __syncthreads();
    if (lane == 0) red[warp] = v;
    __syncthreads();
    float s = 0.f;
    for (int w = 0; w < nw; ++w) s += red[w];            // fixed order: deterministic
    return s;
}

// rotation that annihilates the pivot of a Hermitian 2x2 block [[app, apq],[conj(apq), aqq]]:
// J = [[c, se],[-conj(se), c]], se = s e^{i phi}; identity when the pivot is below thr2 (zero padding too).
// With d = aqq - app:  t = sgn(d) 2|apq| / (|d| + sqrt(d^2 + 4|apq|^2)),  c = 1/sqrt(1+t^2),  se = apq (t/|apq|) c.
// Branch-free and written so that |apq| itself is never needed; the approximate rsqrt / rcp keep the
// dependent chain short.  c^2 + |se|^2 = 1 up to the rounding of one rsqrt, i.e. J is a unitary times
// (1 + O(eps)); the columns of V are renormalised at the end.
__device__ __forceinline__ bool jacobi_rot(float app, float aqq, float2 apq, float thr2, float& c, float2& se) {
    const float mag2 = fmaf(apq.x, apq.x, apq.y * apq.y);
    const bool rot = mag2 > thr2;
    const float d = aqq - app;
    const float x = fmaxf(fmaf(d, d, 4.f * mag2), 1e-36f);
    const float root = x * rsqrt_fast(x);
    const float u = copysignf(2.f, d) * rcp_fast(fabsf(d) + root);      // t / |apq|
    const float cc = rsqrt_fast(fmaf(u * u, mag2, 1.f));
    const float uc = rot ? u * cc : 0.f;
    c = rot ? cc : 1.f;
    se = make_float2(apq.x * uc, apq.y * uc);
    return rot;
}

// position taken in the next step by the row/column now at position pos (round-robin "chairs":
// top row = even positions, bottom row = odd positions, position 0 fixed)
__host__ __device__ constexpr int rr_next(int pos, int Tp) {
    return pos == 0 ? 0 : pos == 1 ? (Tp > 2 ? 2 : 1) : (pos & 1) ? pos - 2 : (pos == Tp - 2 ? Tp - 1 : pos + 2);
}

template <int TP>
__global__ void __launch_bounds__((TP / 2) * (TP / 2) < 32 ? 32 : (TP / 2) * (TP / 2), 1)
k_eig(const float2* __restrict__ C, int T, float* __restrict__ evals, float2* __restrict__ Vout,
      int32_t* __restrict__ status, int max_sweeps, int32_t* __restrict__ noconv) {
    extern __shared__ __align__(16) unsigned char raw[];
    pdl_wait();
    constexpr int Tp = TP, LD = TP + 2, half = TP / 2, m = TP - 1;   // LD even: rows 16-byte aligned for LDS.128
    float2* A0 = reinterpret_cast<float2*>(raw);
    float2* A1 = A0 + Tp * LD;
    float2* V0 = A1 + Tp * LD;
    float2* V1 = V0 + Tp * LD;
    float2* Cs = V1 + Tp * LD;                                      // [T][T] full Hermitian copy of the input
    float* red = reinterpret_cast<float*>(Cs + Tp * Tp);            // [32]
    double* lam = reinterpret_cast<double*>(red + 32);              // [Tp]
    double* dscr = reinterpret_cast<double*>(raw);                  // [T*T], aliases A0/A1 after the sweeps

    const int tid = threadIdx.x, nt = blockDim.x;
    const long long clk0 = clock64();

    // ---- load: lower triangle of C -> full Hermitian Cs; A = Cs scaled by a power of two (max|entry| <= 1); V = I
    float dmax = 0.f;
    for (int i = tid; i < T * T; i += nt) {
        const int r = i / T, c = i - r * T;
        float2 a;
        if (c < r) a = C[i];
        else if (c > r) { a = C[c * T + r]; a.y = -a.y; }
        else a = make_float2(C[i].x, 0.f);
        Cs[i] = a;
        dmax = fmaxf(dmax, fmaxf(fabsf(a.x), fabsf(a.y)));
    }
#pragma unroll
    for (int o = 16; o >= 1; o >>= 1) dmax = fmaxf(dmax, __shfl_xor_sync(0xffffffffu, dmax, o));
    if ((tid & 31) == 0) red[tid >> 5] = dmax;
    __syncthreads();
    dmax = 0.f;
    for (int w = 0; w < (nt >> 5); ++w) dmax = fmaxf(dmax, red[w]);
    int ex = 0;
    if (dmax > 0.f && dmax < 3.0e38f) frexpf(dmax, &ex);
    const float scale = ldexpf(1.f, -ex);
    float n2 = 0.f;
    for (int i = tid; i < Tp * Tp; i += nt) {
        const int r = i / Tp, c = i - r * Tp;
        float2 a = make_float2(0.f, 0.f);
        if (r < T && c < T) { a = Cs[r * T + c]; a.x *= scale; a.y *= scale; }
        A0[r * LD + c] = a;
        V0[r * LD + c] = make_float2(r == c ? 1.f : 0.f, 0.f);
        n2 = fmaf(a.x, a.x, fmaf(a.y, a.y, n2));
    }
    const float normF2 = block_sum(n2, red);
    const float eps = 5.96e-8f;
    const float thr2 = (0.25f * eps * eps / (float)(T * T)) * normF2;   // skip pivots below (eps/2T)*||A||_F
    const float tol2 = (float)(T * T) * eps * eps * normF2;             // stop at off-norm <= T*eps*||A||_F

    // one thread per 2x2 block (pair bi, pair bj) of A; the same thread rotates rows 2bi, 2bi+1 of V by J_bj
    const int bi = tid / half, bj = tid % half;
    const bool worker = tid < half * half;
    const int r0 = 2 * bi, c0 = 2 * bj;
    const int rd0 = rr_next(r0, Tp), rd1 = rr_next(r0 + 1, Tp), cd0 = rr_next(c0, Tp), cd1 = rr_next(c0 + 1, Tp);
    // element offsets (fixed for the whole solve)
    const int oB0 = r0 * LD + c0, oB1 = oB0 + LD;            // block rows (reads, 16-byte vectors)
    const int oDi = r0 * LD + r0, oDj = c0 * LD + c0;        // pivot blocks of pair i and pair j
    const int w00 = rd0 * LD + cd0, w01 = rd0 * LD + cd1, w10 = rd1 * LD + cd0, w11 = rd1 * LD + cd1;
    const int wv00 = r0 * LD + cd0, wv01 = r0 * LD + cd1, wv10 = wv00 + LD, wv11 = wv01 + LD;
    float2 *Ac = A0, *An = A1, *Vc = V0, *Vn = V1;
    int sweeps = 0, converged = 0, last_rot = 0;
    const long long clk1 = clock64();
    for (; sweeps < max_sweeps; ++sweeps) {
        float o2 = 0.f;
        for (int i = tid; i < Tp * Tp; i += nt) {
            const int r = i / Tp, c = i - r * Tp;
            if (r != c) { const float2 a = Ac[r * LD + c]; o2 = fmaf(a.x, a.x, fmaf(a.y, a.y, o2)); }
        }
        const float off2 = block_sum(o2, red);
        if (off2 <= tol2) { converged = 1; break; }
        int applied = 0;
#pragma unroll 1
        for (int step = 0; step < m; ++step) {
            if (worker) {
                // all shared-memory reads of the step are issued before the first use
                const float4 di = *reinterpret_cast<const float4*>(Ac + oDi);       // [app, apq]
                const float aqqi = Ac[oDi + LD + 1].x;
                const float4 dj = *reinterpret_cast<const float4*>(Ac + oDj);
                const float aqqj = Ac[oDj + LD + 1].x;
                const float4 B0 = *reinterpret_cast<const float4*>(Ac + oB0);       // [b00, b01]
                const float4 B1 = *reinterpret_cast<const float4*>(Ac + oB1);       // [b10, b11]
                const float4 U0 = *reinterpret_cast<const float4*>(Vc + oB0);       // V rows r0, r0+1, columns c0, c0+1
                const float4 U1 = *reinterpret_cast<const float4*>(Vc + oB1);
                float ci, cj; float2 sei, sej;
                const bool ri = jacobi_rot(di.x, aqqi, make_float2(di.z, di.w), thr2, ci, sei);
                jacobi_rot(dj.x, aqqj, make_float2(dj.z, dj.w), thr2, cj, sej);
                applied += (bi == bj) && ri;
                const float2 b00 = make_float2(B0.x, B0.y), b01 = make_float2(B0.z, B0.w);
                const float2 b10 = make_float2(B1.x, B1.y), b11 = make_float2(B1.z, B1.w);
                // B' = J_i^H B J_j
                float2 t1, t2;
                t1 = cmulcf(b01, sej); t2 = cmulf(b00, sej);
                const float2 x00 = make_float2(fmaf(cj, b00.x, -t1.x), fmaf(cj, b00.y, -t1.y));
                const float2 x01 = make_float2(fmaf(cj, b01.x, t2.x), fmaf(cj, b01.y, t2.y));
                t1 = cmulcf(b11, sej); t2 = cmulf(b10, sej);
                const float2 x10 = make_float2(fmaf(cj, b10.x, -t1.x), fmaf(cj, b10.y, -t1.y));
                const float2 x11 = make_float2(fmaf(cj, b11.x, t2.x), fmaf(cj, b11.y, t2.y));
                t1 = cmulf(x10, sei); t2 = cmulcf(x00, sei);
                float2 y00 = make_float2(fmaf(ci, x00.x, -t1.x), fmaf(ci, x00.y, -t1.y));
                float2 y10 = make_float2(fmaf(ci, x10.x, t2.x), fmaf(ci, x10.y, t2.y));
                t1 = cmulf(x11, sei); t2 = cmulcf(x01, sei);
                float2 y01 = make_float2(fmaf(ci, x01.x, -t1.x), fmaf(ci, x01.y, -t1.y));
                float2 y11 = make_float2(fmaf(ci, x11.x, t2.x), fmaf(ci, x11.y, t2.y));
                if (bi == bj) {                      // the pivot block: exactly diagonal and real afterwards
                    y00.y = 0.f; y11.y = 0.f;
                    if (ri) { y01 = make_float2(0.f, 0.f); y10 = make_float2(0.f, 0.f); }
                }
                An[w00] = y00; An[w01] = y01; An[w10] = y10; An[w11] = y11;
                // V <- V J_j on rows r0, r0+1
                const float2 v0p = make_float2(U0.x, U0.y), v0q = make_float2(U0.z, U0.w);
                const float2 v1p = make_float2(U1.x, U1.y), v1q = make_float2(U1.z, U1.w);
                t1 = cmulcf(v0q, sej); t2 = cmulf(v0p, sej);
                Vn[wv00] = make_float2(fmaf(cj, v0p.x, -t1.x), fmaf(cj, v0p.y, -t1.y));
                Vn[wv01] = make_float2(fmaf(cj, v0q.x, t2.x), fmaf(cj, v0q.y, t2.y));
                t1 = cmulcf(v1q, sej); t2 = cmulf(v1p, sej);
                Vn[wv10] = make_float2(fmaf(cj, v1p.x, -t1.x), fmaf(cj, v1p.y, -t1.y));
                Vn[wv11] = make_float2(fmaf(cj, v1q.x, t2.x), fmaf(cj, v1q.y, t2.y));
            }
            __syncthreads();
            float2* tmp = Ac; Ac = An; An = tmp;
            tmp = Vc; Vc = Vn; Vn = tmp;
        }
        last_rot = (int)(block_sum((float)applied, red) + 0.5f);      // rotations applied in this sweep (<= Tp^2/2: exact)
        if (last_rot == 0) { converged = 1; ++sweeps; break; }
    }
    __syncthreads();
    const long long clk2 = clock64();
    // m steps of the chair permutation are the identity, so after whole sweeps position == original index
    const float2* V = Vc;

    // ---- FP64 Rayleigh quotients against the original C (shared-memory copy), FP32 vectors
    // (A0/A1 are dead: dscr aliases them; V0/V1/Cs are not touched)
    // thread = (column k, row group); RB rows of C share every load of v_sk
    {
        constexpr int RB = 4;
        const int k = tid % T, g = tid / T, ng = nt / T > 0 ? nt / T : 1;
        for (int tb = g * RB; tb < T && tid < ng * T; tb += ng * RB) {
            double wr[RB], wi[RB];
#pragma unroll
            for (int j = 0; j < RB; ++j) { wr[j] = 0.0; wi[j] = 0.0; }
            for (int s = 0; s < T; ++s) {
                const float2 v = V[s * LD + k];
                const double vx = (double)v.x, vy = (double)v.y;
#pragma unroll
                for (int j = 0; j < RB; ++j) {
                    const int t = min(tb + j, T - 1);
                    const float2 cf = Cs[t * T + s];
                    wr[j] += (double)cf.x * vx - (double)cf.y * vy;
                    wi[j] += (double)cf.x * vy + (double)cf.y * vx;
                }
            }
#pragma unroll
            for (int j = 0; j < RB; ++j) {
                const int t = tb + j;
                if (t < T) { const float2 vt = V[t * LD + k]; dscr[t * T + k] = (double)vt.x * wr[j] + (double)vt.y * wi[j]; }   // Re(conj(v_tk) w_tk)
            }
        }
    }
    __syncthreads();
    if (tid < T) {
        double l = 0.0, nn = 0.0;
        for (int t = 0; t < T; ++t) { l += dscr[t * T + tid]; const float2 v = V[t * LD + tid]; nn += (double)v.x * v.x + (double)v.y * v.y; }
        lam[tid] = nn > 0.0 ? l / nn : 0.0;
    }
    __syncthreads();
    if (tid < T) {
        const double l = lam[tid];
        int r = 0;
        for (int j = 0; j < T; ++j) { const double lj = lam[j]; r += (lj > l) || (lj == l && j < tid); }
        // normalise + canonical phase
        float best = -1.f; float2 bv = make_float2(1.f, 0.f); float nn = 0.f;
        for (int t = 0; t < T; ++t) {
            const float2 v = V[t * LD + tid];
            const float a2 = v.x * v.x + v.y * v.y;
            nn += a2;
            if (a2 > best) { best = a2; bv = v; }
        }
        const float inv = (best > 0.f) ? 1.f / (sqrtf(best) * sqrtf(nn)) : 1.f;
        const float2 ph = make_float2(bv.x * inv, -bv.y * inv);    // conj(bv)/(|bv| ||v||)
        for (int t = 0; t < T; ++t) Vout[t * T + r] = cmulf(V[t * LD + tid], ph);
        evals[r] = (float)l;
    }
    if (tid == 0) {
        status[0] = converged ? 0 : 1;
        status[1] = sweeps;
        status[2] = last_rot;
        status[3] = 0;
        status[4] = (int)(clk1 - clk0);          // cycles: load + scale
        status[5] = (int)(clk2 - clk1);          // cycles: Jacobi sweeps
        status[6] = (int)(clock64() - clk2);     // cycles: Rayleigh refinement, sort, phase fix
        status[7] = 0;
        // sticky host-visible flag (mapped pinned word): the next API call on the handle returns HOLO_ERR_NOCONV
        if (!converged && noconv) { *(volatile int32_t*)noconv = 1; __threadfence_system(); }
    }
}

// ------------------------------------------------------------------------------------------------
// Real symmetric form of the same solver.  Inside holo_process / holo_submit / holo_push the covariance is real
// symmetric in exact arithmetic (R21: holograms of real frames; exactly so when it comes from the integer Gram
// of the raw frames), and it is stored with Im = 0: rotations, updates and eigenvectors are then real, the step body is
// 60 % of the complex one (it is bound by instruction issue: one thread per 2x2 block, two rotations per thread) and
// the shared-memory footprint is halved.  Same ordering, thresholds, FP64 refinement, sorting and sign convention
// (largest-magnitude entry positive), same status words.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ bool jacobi_rot_real(float app, float aqq, float apq, float thr2, float& c, float& s) {
    const float mag2 = apq * apq;
    const bool rot = mag2 > thr2;
    const float d = aqq - app;
    const float x = fmaxf(fmaf(d, d, 4.f * mag2), 1e-36f);
    const float root = x * rsqrt_fast(x);
    const float u = copysignf(2.f, d) * rcp_fast(fabsf(d) + root);      // t / |apq|
    const float cc = rsqrt_fast(fmaf(u * u, mag2, 1.f));
    const float uc = rot ? u * cc : 0.f;
    c = rot ? cc : 1.f;
    s = apq * uc;
    return rot;
}

template <int TP>
__global__ void __launch_bounds__((TP / 2) * (TP / 2) < 32 ? 32 : (TP / 2) * (TP / 2), 1)
k_eig_real(const float2* __restrict__ C, int T, float* __restrict__ evals, float2* __restrict__ Vout,
           int32_t* __restrict__ status, int max_sweeps, int32_t* __restrict__ noconv) {
    extern __shared__ __align__(16) unsigned char raw[];
    pdl_wait();                                                     // (launched as a programmatic dependent of the reduction)
    constexpr int Tp = TP, LD = TP + 2, half = TP / 2, m = TP - 1;   // LD even: pairs 8-byte aligned
    float* A0 = reinterpret_cast<float*>(raw);
    float* A1 = A0 + Tp * LD;
    float* V0 = A1 + Tp * LD;
    float* V1 = V0 + Tp * LD;
    float* Cs = V1 + Tp * LD;                                       // [T][T] full symmetric copy of the input
    float* red = Cs + Tp * Tp;                                      // [32]
    double* lam = reinterpret_cast<double*>(red + 32);              // [Tp]
    double* dscr = lam + Tp;                                        // [T*T]

    const int tid = threadIdx.x, nt = blockDim.x;
    const long long clk0 = clock64();
    float dmax = 0.f;
    for (int i = tid; i < T * T; i += nt) {
        const int r = i / T, c = i - r * T;
        const float a = c <= r ? C[i].x : C[c * T + r].x;           // lower triangle
        Cs[i] = a;
        dmax = fmaxf(dmax, fabsf(a));
    }
#pragma unroll
    for (int o = 16; o >= 1; o >>= 1) dmax = fmaxf(dmax, __shfl_xor_sync(0xffffffffu, dmax, o));
    if ((tid & 31) == 0) red[tid >> 5] = dmax;
    __syncthreads();
    dmax = 0.f;
    for (int w = 0; w < (nt >> 5); ++w) dmax = fmaxf(dmax, red[w]);
    int ex = 0;
    if (dmax > 0.f && dmax < 3.0e38f) frexpf(dmax, &ex);
    const float scale = ldexpf(1.f, -ex);
    float n2 = 0.f;
    for (int i = tid; i < Tp * Tp; i += nt) {
        const int r = i / Tp, c = i - r * Tp;
        float a = 0.f;
        if (r < T && c < T) a = Cs[r * T + c] * scale;
        A0[r * LD + c] = a;
        V0[r * LD + c] = r == c ? 1.f : 0.f;
        n2 = fmaf(a, a, n2);
    }
    const float normF2 = block_sum(n2, red);
    const float eps = 5.96e-8f;
    const float thr2 = (0.25f * eps * eps / (float)(T * T)) * normF2;
    const float tol2 = (float)(T * T) * eps * eps * normF2;

    const int bi = tid / half, bj = tid % half;
    const bool worker = tid < half * half;
    const int r0 = 2 * bi, c0 = 2 * bj;
    const int rd0 = rr_next(r0, Tp), rd1 = rr_next(r0 + 1, Tp), cd0 = rr_next(c0, Tp), cd1 = rr_next(c0 + 1, Tp);
    const int oB0 = r0 * LD + c0, oB1 = oB0 + LD;
    const int oDi = r0 * LD + r0, oDj = c0 * LD + c0;
    const int w00 = rd0 * LD + cd0, w01 = rd0 * LD + cd1, w10 = rd1 * LD + cd0, w11 = rd1 * LD + cd1;
    const int wv00 = r0 * LD + cd0, wv01 = r0 * LD + cd1, wv10 = wv00 + LD, wv11 = wv01 + LD;
    float *Ac = A0, *An = A1, *Vc = V0, *Vn = V1;
    int sweeps = 0, converged = 0, last_rot = 0;
    const long long clk1 = clock64();
    for (; sweeps < max_sweeps; ++sweeps) {
        float o2 = 0.f;
        for (int i = tid; i < Tp * Tp; i += nt) {
            const int r = i / Tp, c = i - r * Tp;
            if (r != c) { const float a = Ac[r * LD + c]; o2 = fmaf(a, a, o2); }
        }
        const float off2 = block_sum(o2, red);
        if (off2 <= tol2) { converged = 1; break; }
        int applied = 0;
#pragma unroll 1
        for (int step = 0; step < m; ++step) {
            if (worker) {
                const float2 di = *reinterpret_cast<const float2*>(Ac + oDi);       // [app, apq]
                const float aqqi = Ac[oDi + LD + 1];
                const float2 dj = *reinterpret_cast<const float2*>(Ac + oDj);
                const float aqqj = Ac[oDj + LD + 1];
                const float2 B0 = *reinterpret_cast<const float2*>(Ac + oB0);       // [b00, b01]
                const float2 B1 = *reinterpret_cast<const float2*>(Ac + oB1);       // [b10, b11]
                const float2 U0 = *reinterpret_cast<const float2*>(Vc + oB0);
                const float2 U1 = *reinterpret_cast<const float2*>(Vc + oB1);
                float ci, cj, si, sj;
                const bool ri = jacobi_rot_real(di.x, aqqi, di.y, thr2, ci, si);
                jacobi_rot_real(dj.x, aqqj, dj.y, thr2, cj, sj);
                applied += (bi == bj) && ri;
                // B' = J_i^T B J_j,  J = [[c, s], [-s, c]]
                const float x00 = fmaf(cj, B0.x, -sj * B0.y), x01 = fmaf(cj, B0.y, sj * B0.x);
                const float x10 = fmaf(cj, B1.x, -sj * B1.y), x11 = fmaf(cj, B1.y, sj * B1.x);
                float y00 = fmaf(ci, x00, -si * x10), y10 = fmaf(ci, x10, si * x00);
                float y01 = fmaf(ci, x01, -si * x11), y11 = fmaf(ci, x11, si * x01);
                if (bi == bj && ri) { y01 = 0.f; y10 = 0.f; }                       // the pivot block: exactly diagonal afterwards
                An[w00] = y00; An[w01] = y01; An[w10] = y10; An[w11] = y11;
                Vn[wv00] = fmaf(cj, U0.x, -sj * U0.y); Vn[wv01] = fmaf(cj, U0.y, sj * U0.x);
                Vn[wv10] = fmaf(cj, U1.x, -sj * U1.y); Vn[wv11] = fmaf(cj, U1.y, sj * U1.x);
            }
            __syncthreads();
            float* tmp = Ac; Ac = An; An = tmp;
            tmp = Vc; Vc = Vn; Vn = tmp;
        }
        last_rot = (int)(block_sum((float)applied, red) + 0.5f);
        if (last_rot == 0) { converged = 1; ++sweeps; break; }
    }
    __syncthreads();
    const long long clk2 = clock64();
    const float* V = Vc;
    {   // FP64 Rayleigh quotients against the original C
        constexpr int RB = 4;
        const int k = tid % T, g = tid / T, ng = nt / T > 0 ? nt / T : 1;
        for (int tb = g * RB; tb < T && tid < ng * T; tb += ng * RB) {
            double wr[RB];
#pragma unroll
            for (int j = 0; j < RB; ++j) wr[j] = 0.0;
            for (int s = 0; s < T; ++s) {
                const double vx = (double)V[s * LD + k];
#pragma unroll
                for (int j = 0; j < RB; ++j) wr[j] += (double)Cs[min(tb + j, T - 1) * T + s] * vx;
            }
#pragma unroll
            for (int j = 0; j < RB; ++j) {
                const int t = tb + j;
                if (t < T) dscr[t * T + k] = (double)V[t * LD + k] * wr[j];
            }
        }
    }
    __syncthreads();
    if (tid < T) {
        double l = 0.0, nn = 0.0;
        for (int t = 0; t < T; ++t) { l += dscr[t * T + tid]; const double v = (double)V[t * LD + tid]; nn += v * v; }
        lam[tid] = nn > 0.0 ? l / nn : 0.0;
    }
    __syncthreads();
    if (tid < T) {
        const double l = lam[tid];
        int r = 0;
        for (int j = 0; j < T; ++j) { const double lj = lam[j]; r += (lj > l) || (lj == l && j < tid); }
        float best = -1.f, bv = 1.f, nn = 0.f;
        for (int t = 0; t < T; ++t) {
            const float v = V[t * LD + tid];
            const float a2 = v * v;
            nn += a2;
            if (a2 > best) { best = a2; bv = v; }
        }
        const float sgn = (best > 0.f) ? copysignf(1.f / sqrtf(nn), bv) : 1.f;      // normalise, largest-magnitude entry positive
        for (int t = 0; t < T; ++t) Vout[t * T + r] = make_float2(V[t * LD + tid] * sgn, 0.f);
        evals[r] = (float)l;
    }
    if (tid == 0) {
        status[0] = converged ? 0 : 1;
        status[1] = sweeps;
        status[2] = last_rot;
        status[3] = 0;
        status[4] = (int)(clk1 - clk0);
        status[5] = (int)(clk2 - clk1);
        status[6] = (int)(clock64() - clk2);
        status[7] = 0;
        if (!converged && noconv) { *(volatile int32_t*)noconv = 1; __threadfence_system(); }
    }
}

template <int TP>
static int launch_eig_real_t(holo_ctx* c, const float2* C, float* evals, float2* V, cudaStream_t st) {
    const int T = c->T;
    constexpr int LD = TP + 2;
    constexpr size_t smem = (size_t)4 * TP * LD * sizeof(float) + (size_t)TP * TP * sizeof(float) + 32 * sizeof(float)
                          + TP * sizeof(double) + (size_t)TP * TP * sizeof(double);
    { const int rc = holo_ensure_smem_attr((const void*)k_eig_real<TP>, c->device, smem); if (rc) return rc; }
    constexpr int threads = (TP / 2) * (TP / 2) < 32 ? 32 : (TP / 2) * (TP / 2);
    HoloProf prof(c, HOLO_K_EIG, st);
    HOLO_CUDA_OK(holo_launch_pdl(k_eig_real<TP>, dim3(1), dim3(threads), smem, st, C, T, evals, V, c->status, c->tune[HOLO_TUNE_EIG_MAX_SWEEPS], c->noconv_dev));
    HOLO_CUDA_OK(cudaGetLastError());
    return HOLO_OK;
}

template <int TP>
static int launch_eig_t(holo_ctx* c, const float2* C, float* evals, float2* V, cudaStream_t st) {
    const int T = c->T;
    constexpr int LD = TP + 2;
    // A0, A1, V0, V1 [TP][LD] + Cs [TP][TP] float2, red[32] float, lam[TP] double
    constexpr size_t smem = (size_t)4 * TP * LD * sizeof(float2) + (size_t)TP * TP * sizeof(float2) + 32 * sizeof(float)
                          + TP * sizeof(double);
    { const int rc = holo_ensure_smem_attr((const void*)k_eig<TP>, c->device, smem); if (rc) return rc; }
    constexpr int threads = (TP / 2) * (TP / 2) < 32 ? 32 : (TP / 2) * (TP / 2);
    HoloProf prof(c, HOLO_K_EIG, st);
    HOLO_CUDA_OK(holo_launch_pdl(k_eig<TP>, dim3(1), dim3(threads), smem, st, C, T, evals, V, c->status, c->tune[HOLO_TUNE_EIG_MAX_SWEEPS], c->noconv_dev));
    HOLO_CUDA_OK(cudaGetLastError());
    return HOLO_OK;
}

int holo_launch_eig(holo_ctx* c, const float2* C, float* evals, float2* V, cudaStream_t st, bool real_symmetric) {
    const int T = c->T;
    if (real_symmetric) {
        if (T <= 4) return launch_eig_real_t<4>(c, C, evals, V, st);
        if (T <= 8) return launch_eig_real_t<8>(c, C, evals, V, st);
        if (T <= 16) return launch_eig_real_t<16>(c, C, evals, V, st);
        if (T <= 32) return launch_eig_real_t<32>(c, C, evals, V, st);
        return launch_eig_real_t<64>(c, C, evals, V, st);
    }
    if (T <= 4) return launch_eig_t<4>(c, C, evals, V, st);
    if (T <= 8) return launch_eig_t<8>(c, C, evals, V, st);
    if (T <= 16) return launch_eig_t<16>(c, C, evals, V, st);
    if (T <= 32) return launch_eig_t<32>(c, C, evals, V, st);
    return launch_eig_t<64>(c, C, evals, V, st);
}
