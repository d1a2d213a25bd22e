// eig.cu -- A4: C = V Lambda V^{t*}   (Eq. 5; R1 descending order, R8, R10, R11)
//
// Single-CTA two-sided complex Hermitian Jacobi in FP32, parallel (round-robin tournament) ordering:
// each of the Tp-1 steps of a sweep annihilates Tp/2 disjoint pivots at once.  A and V live in
// shared memory.  After convergence the eigenvalues are refined as FP64 Rayleigh quotients
// v_k^H C v_k of the ORIGINAL matrix, sorted descending, and every eigenvector is normalised and
// phase-fixed (largest-magnitude entry real positive, ties -> lowest index).
#include "holo_internal.cuh"

__device__ __forceinline__ float2 cmulf(float2 a, float2 b) {
    return make_float2(fmaf(-a.y, b.y, a.x * b.x), fmaf(a.y, b.x, a.x * b.y));
}
__device__ __forceinline__ float2 cmulcf(float2 a, float2 b) {      // a * conj(b)
    return make_float2(fmaf(a.y, b.y, a.x * b.x), fmaf(a.y, b.x, -a.x * b.y));
}

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
// J = [[c, se],[-conj(se), c]], se = s e^{i phi}; identity when the pivot is below thr2 (or padding).
__device__ __forceinline__ bool jacobi_rot(float app, float aqq, float2 apq, float thr2, bool valid, float& c, float2& se) {
    c = 1.f; se = make_float2(0.f, 0.f);
    const float mag2 = fmaf(apq.x, apq.x, apq.y * apq.y);
    if (!valid || !(mag2 > thr2)) return false;
    const float inv_mag = rsqrtf(mag2);
    const float m2 = 2.f * mag2 * inv_mag;                  // 2|apq|
    const float d = aqq - app;
    const float t = copysignf(m2, d) / (fabsf(d) + sqrtf(fmaf(d, d, m2 * m2)));   // sgn(tau)/(|tau|+sqrt(1+tau^2))
    c = rsqrtf(fmaf(t, t, 1.f));
    const float s = t * c * inv_mag;
    se = make_float2(apq.x * s, apq.y * s);
    return true;
}

template <int TP>
__global__ void __launch_bounds__((TP / 2) * (TP / 2) < 32 ? 32 : (TP / 2) * (TP / 2), 1)
k_eig(const float2* __restrict__ C, int T, float* __restrict__ evals, float2* __restrict__ Vout,
      int32_t* __restrict__ status, int max_sweeps) {
    extern __shared__ __align__(16) unsigned char raw[];
    constexpr int Tp = TP, LD = TP + 1, half = TP / 2, m = TP - 1;
    float2* A0 = reinterpret_cast<float2*>(raw);
    float2* A1 = A0 + Tp * LD;
    float2* V = A1 + Tp * LD;
    float* red = reinterpret_cast<float*>(V + Tp * LD);             // [32]
    size_t off = (size_t)((unsigned char*)(red + 32) - raw);
    off = (off + 15) & ~(size_t)15;
    double* dscr = reinterpret_cast<double*>(raw + off);            // [T*T] partial Rayleigh terms
    double* lam = dscr + (size_t)T * T;                             // [T]
    int* rank = reinterpret_cast<int*>(lam + T);                    // [T]

    const int tid = threadIdx.x, nt = blockDim.x;
    const long long clk0 = clock64();

    // ---- load: lower triangle of C -> full Hermitian A (scaled by a power of two so that max|diag| <= 1); V = I
    float dmax = 0.f;
    for (int i = tid; i < T; i += nt) dmax = fmaxf(dmax, fabsf(C[i * T + i].x));
    for (int i = tid; i < T * T; i += nt) { const int r = i / T, c = i - r * T; if (c < r) { const float2 a = C[i]; dmax = fmaxf(dmax, fmaxf(fabsf(a.x), fabsf(a.y))); } }
#pragma unroll
    for (int o = 16; o >= 1; o >>= 1) dmax = fmaxf(dmax, __shfl_xor_sync(0xffffffffu, dmax, o));
    if ((tid & 31) == 0) red[tid >> 5] = dmax;
    __syncthreads();
    dmax = 0.f;
    for (int w = 0; w < (nt >> 5); ++w) dmax = fmaxf(dmax, red[w]);
    int ex = 0;
    if (dmax > 0.f && dmax < 3.0e38f) frexpf(dmax, &ex);
    const float scale = ldexpf(1.f, -ex);
    for (int i = tid; i < Tp * Tp; i += nt) {
        const int r = i / Tp, c = i - r * Tp;
        float2 a = make_float2(0.f, 0.f);
        if (r < T && c < T) {
            if (c < r) a = C[r * T + c];
            else if (c > r) { a = C[c * T + r]; a.y = -a.y; }
            else a = make_float2(C[r * T + r].x, 0.f);
            a.x *= scale; a.y *= scale;
        }
        A0[r * LD + c] = a;
        V[r * LD + c] = make_float2(r == c ? 1.f : 0.f, 0.f);
    }
    __syncthreads();
    float n2 = 0.f;
    for (int i = tid; i < Tp * Tp; i += nt) { const float2 a = A0[(i / Tp) * LD + (i % Tp)]; n2 += a.x * a.x + a.y * a.y; }
    const float normF2 = block_sum(n2, red);
    const float eps = 5.96e-8f;
    const float thr2 = (0.25f * eps * eps / (float)(T * T)) * normF2;   // skip pivots below (eps/2T)*||A||_F
    const float tol2 = (float)(T * T) * eps * eps * normF2;             // stop at off-norm <= T*eps*||A||_F

    // one thread per 2x2 block (pair bi, pair bj) of A; the same thread rotates rows 2bi, 2bi+1 of V by J_bj
    const int bi = tid / half, bj = tid % half;
    const bool worker = tid < half * half;
    float2* Ac = A0;
    float2* An = A1;
    int sweeps = 0, converged = 0, last_rot = 0;
    const long long clk1 = clock64();
    for (; sweeps < max_sweeps; ++sweeps) {
        float o2 = 0.f;
        for (int i = tid; i < Tp * Tp; i += nt) {
            const int r = i / Tp, c = i - r * Tp;
            if (r != c) { const float2 a = Ac[r * LD + c]; o2 += a.x * a.x + a.y * a.y; }
        }
        const float off2 = block_sum(o2, red);
        if (off2 <= tol2) { converged = 1; break; }
        int rot_count = 0;
#pragma unroll 1
        for (int step = 0; step < m; ++step) {
            int applied = 0;
            if (worker) {
                int pi, qi, pj, qj;
                if (bi == 0) { pi = step; qi = m; } else { const int a = (step + bi) % m, b = (step - bi + m) % m; pi = min(a, b); qi = max(a, b); }
                if (bj == 0) { pj = step; qj = m; } else { const int a = (step + bj) % m, b = (step - bj + m) % m; pj = min(a, b); qj = max(a, b); }
                float ci, cj; float2 sei, sej;
                const bool ri = jacobi_rot(Ac[pi * LD + pi].x, Ac[qi * LD + qi].x, Ac[pi * LD + qi], thr2, qi < T, ci, sei);
                jacobi_rot(Ac[pj * LD + pj].x, Ac[qj * LD + qj].x, Ac[pj * LD + qj], thr2, qj < T, cj, sej);
                applied = (bi == bj) && ri;
                // B' = J_i^H B J_j
                const float2 b00 = Ac[pi * LD + pj], b01 = Ac[pi * LD + qj], b10 = Ac[qi * LD + pj], b11 = Ac[qi * LD + qj];
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
                An[pi * LD + pj] = y00; An[pi * LD + qj] = y01; An[qi * LD + pj] = y10; An[qi * LD + qj] = y11;
                // V <- V J_j on rows 2bi, 2bi+1 (in place: nobody else touches these elements this step)
#pragma unroll
                for (int rr = 0; rr < 2; ++rr) {
                    const int r = 2 * bi + rr;
                    const float2 vp = V[r * LD + pj], vq = V[r * LD + qj];
                    t1 = cmulcf(vq, sej); t2 = cmulf(vp, sej);
                    V[r * LD + pj] = make_float2(fmaf(cj, vp.x, -t1.x), fmaf(cj, vp.y, -t1.y));
                    V[r * LD + qj] = make_float2(fmaf(cj, vq.x, t2.x), fmaf(cj, vq.y, t2.y));
                }
            }
            rot_count += __syncthreads_count(applied);
            float2* tmp = Ac; Ac = An; An = tmp;
        }
        last_rot = rot_count;
        if (last_rot == 0) { converged = 1; ++sweeps; break; }
    }
    __syncthreads();
    const long long clk2 = clock64();

    // ---- FP64 Rayleigh quotients against the original C (Hermitian from its lower triangle)
    for (int i = tid; i < T * T; i += nt) {
        const int t = i / T, k = i - t * T;
        double wr = 0.0, wi = 0.0;
        for (int s = 0; s < T; ++s) {
            float2 cf;
            if (s < t) cf = C[t * T + s];
            else if (s > t) { cf = C[s * T + t]; cf.y = -cf.y; }
            else cf = make_float2(C[t * T + t].x, 0.f);
            const float2 v = V[s * LD + k];
            wr += (double)cf.x * v.x - (double)cf.y * v.y;
            wi += (double)cf.x * v.y + (double)cf.y * v.x;
        }
        const float2 vt = V[t * LD + k];
        dscr[i] = (double)vt.x * wr + (double)vt.y * wi;          // Re(conj(v_tk) w_tk)
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
        rank[tid] = r;
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
    }
}

template <int TP>
static int launch_eig_t(holo_ctx* c, const float2* C, float* evals, float2* V, cudaStream_t st) {
    const int T = c->T;
    constexpr int LD = TP + 1;
    size_t smem = (size_t)3 * TP * LD * sizeof(float2) + 32 * sizeof(float);
    smem = (smem + 15) & ~(size_t)15;
    smem += (size_t)T * T * sizeof(double) + T * sizeof(double) + T * sizeof(int) + 16;
    static bool attr = false;
    if (!attr) {
        const size_t worst = (size_t)3 * TP * LD * sizeof(float2) + 256 + (size_t)TP * TP * 8 + TP * 12 + 32;
        HOLO_CUDA_OK(cudaFuncSetAttribute(k_eig<TP>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)worst));
        attr = true;
    }
    constexpr int threads = (TP / 2) * (TP / 2) < 32 ? 32 : (TP / 2) * (TP / 2);
    HoloProf prof(c, HOLO_K_EIG, st);
    k_eig<TP><<<1, threads, smem, st>>>(C, T, evals, V, c->status, c->tune[HOLO_TUNE_EIG_MAX_SWEEPS]);
    HOLO_CUDA_OK(cudaGetLastError());
    return HOLO_OK;
}

int holo_launch_eig(holo_ctx* c, const float2* C, float* evals, float2* V, cudaStream_t st) {
    const int T = c->T;
    if (T <= 4) return launch_eig_t<4>(c, C, evals, V, st);
    if (T <= 8) return launch_eig_t<8>(c, C, evals, V, st);
    if (T <= 16) return launch_eig_t<16>(c, C, evals, V, st);
    if (T <= 32) return launch_eig_t<32>(c, C, evals, V, st);
    return launch_eig_t<64>(c, C, evals, V, st);
}
