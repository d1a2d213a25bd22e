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

__global__ void __launch_bounds__(512, 1)
k_eig(const float2* __restrict__ C, int T, float* __restrict__ evals, float2* __restrict__ Vout,
      int32_t* __restrict__ status, int max_sweeps) {
    extern __shared__ __align__(16) unsigned char raw[];
    const int Tp = (T + 1) & ~1;
    const int LD = Tp + 1;
    float2* A = reinterpret_cast<float2*>(raw);
    float2* V = A + Tp * LD;
    float2* rot_se = V + Tp * LD;                 // [Tp/2] s*e^{i phi}
    float* rot_c = reinterpret_cast<float*>(rot_se + Tp / 2);       // [Tp/2]
    int* rot_p = reinterpret_cast<int*>(rot_c + Tp / 2);
    int* rot_q = rot_p + Tp / 2;
    float* red = reinterpret_cast<float*>(rot_q + Tp / 2);          // [32]
    int* cnt = reinterpret_cast<int*>(red + 32);                    // [2]
    size_t off = (size_t)((unsigned char*)(cnt + 2) - raw);
    off = (off + 15) & ~(size_t)15;
    double* dscr = reinterpret_cast<double*>(raw + off);            // [T*T] partial Rayleigh terms
    double* lam = dscr + (size_t)T * T;                             // [T]
    int* rank = reinterpret_cast<int*>(lam + T);                    // [T]

    const int tid = threadIdx.x, nt = blockDim.x;
    const int half = Tp / 2, m = Tp - 1;

    // ---- load: lower triangle of C -> full Hermitian A; V = I
    for (int i = tid; i < Tp * Tp; i += nt) {
        int r = i / Tp, c = i - r * Tp;
        float2 a = make_float2(0.f, 0.f);
        if (r < T && c < T) {
            if (c < r) a = C[r * T + c];
            else if (c > r) { a = C[c * T + r]; a.y = -a.y; }
            else a = make_float2(C[r * T + r].x, 0.f);
        }
        A[r * LD + c] = a;
        V[r * LD + c] = make_float2(r == c ? 1.f : 0.f, 0.f);
    }
    if (tid == 0) { cnt[0] = 0; cnt[1] = 0; }
    __syncthreads();
    float n2 = 0.f;
    for (int i = tid; i < Tp * Tp; i += nt) { float2 a = A[(i / Tp) * LD + (i % Tp)]; n2 += a.x * a.x + a.y * a.y; }
    const float normF2 = block_sum(n2, red);
    const float eps = 5.96e-8f;
    const float thr2 = (0.25f * eps * eps / (float)(T * T)) * normF2;   // skip pivots below (eps/2T)*||A||_F
    const float tol2 = (float)(T * T) * eps * eps * normF2;             // stop at off-norm <= T*eps*||A||_F

    int sweeps = 0, converged = 0, last_rot = 0;
    for (; sweeps < max_sweeps; ++sweeps) {
        if (tid == 0) cnt[0] = 0;            // ordered before the pivots' atomicAdd by block_sum's barriers
        float o2 = 0.f;
        for (int i = tid; i < Tp * Tp; i += nt) {
            int r = i / Tp, c = i - r * Tp;
            if (r != c) { float2 a = A[r * LD + c]; o2 += a.x * a.x + a.y * a.y; }
        }
        const float off2 = block_sum(o2, red);
        if (off2 <= tol2) { converged = 1; break; }
        for (int step = 0; step < m; ++step) {
            // ---- 1. rotations for the Tp/2 disjoint pivots of this step
            if (tid < half) {
                int p, q;
                if (tid == 0) { p = step; q = m; }
                else { int a = (step + tid) % m, b = (step - tid + m) % m; p = a < b ? a : b; q = a < b ? b : a; }
                float c = 1.f; float2 se = make_float2(0.f, 0.f);
                if (q < T) {
                    const float2 apq = A[p * LD + q];
                    const float mag2 = apq.x * apq.x + apq.y * apq.y;
                    if (mag2 > thr2 && mag2 > 0.f) {
                        const float app = A[p * LD + p].x, aqq = A[q * LD + q].x;
                        const float mag = sqrtf(mag2);
                        const float tau = (aqq - app) / (2.f * mag);
                        const float t = copysignf(1.f, tau) / (fabsf(tau) + sqrtf(fmaf(tau, tau, 1.f)));
                        c = 1.f / sqrtf(fmaf(t, t, 1.f));
                        const float s = t * c, inv = s / mag;
                        se = make_float2(apq.x * inv, apq.y * inv);
                        atomicAdd(&cnt[0], 1);
                    }
                }
                rot_c[tid] = c; rot_se[tid] = se; rot_p[tid] = p; rot_q[tid] = q;
            }
            __syncthreads();
            // ---- 2. A <- A J, V <- V J   (columns p,q; lanes run over rows: stride LD is odd -> no conflicts)
            for (int i = tid; i < 2 * half * Tp; i += nt) {
                const int row = i % Tp, pr = (i / Tp) % half, which = i / (Tp * half);
                float2* M = which ? V : A;
                const int p = rot_p[pr], q = rot_q[pr];
                const float c = rot_c[pr]; const float2 se = rot_se[pr];
                const float2 ap = M[row * LD + p], aq = M[row * LD + q];
                const float2 t1 = cmulcf(aq, se);          // aq * s e^{-i phi}
                const float2 t2 = cmulf(ap, se);           // ap * s e^{+i phi}
                M[row * LD + p] = make_float2(fmaf(c, ap.x, -t1.x), fmaf(c, ap.y, -t1.y));
                M[row * LD + q] = make_float2(fmaf(c, aq.x, t2.x), fmaf(c, aq.y, t2.y));
            }
            __syncthreads();
            // ---- 3. A <- J^H A   (rows p,q; lanes run over columns)
            for (int i = tid; i < half * Tp; i += nt) {
                const int col = i % Tp, pr = i / Tp;
                const int p = rot_p[pr], q = rot_q[pr];
                const float c = rot_c[pr]; const float2 se = rot_se[pr];
                const float2 ap = A[p * LD + col], aq = A[q * LD + col];
                const float2 t1 = cmulf(aq, se);           // s e^{+i phi} aq
                const float2 t2 = cmulcf(ap, se);          // s e^{-i phi} ap
                A[p * LD + col] = make_float2(fmaf(c, ap.x, -t1.x), fmaf(c, ap.y, -t1.y));
                A[q * LD + col] = make_float2(fmaf(c, aq.x, t2.x), fmaf(c, aq.y, t2.y));
            }
            __syncthreads();
        }
        last_rot = cnt[0];
        if (last_rot == 0) { converged = 1; ++sweeps; break; }
        __syncthreads();
    }

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
    }
}

static size_t eig_smem_bytes(int T) {
    const int Tp = (T + 1) & ~1, LD = Tp + 1, half = Tp / 2;
    size_t b = (size_t)2 * Tp * LD * sizeof(float2) + half * (sizeof(float2) + sizeof(float) + 2 * sizeof(int)) +
               32 * sizeof(float) + 2 * sizeof(int);
    b = (b + 15) & ~(size_t)15;
    b += (size_t)T * T * sizeof(double) + T * sizeof(double) + T * sizeof(int);
    return b + 16;
}

int holo_launch_eig(holo_ctx* c, const float2* C, float* evals, float2* V, cudaStream_t st) {
    const size_t smem = eig_smem_bytes(c->T);
    static size_t attr_set = 0;
    if (smem > attr_set) {
        HOLO_CUDA_OK(cudaFuncSetAttribute(k_eig, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        attr_set = smem;
    }
    const int threads = c->T <= 32 ? 256 : 512;
    HoloProf prof(c, HOLO_K_EIG, st);
    k_eig<<<1, threads, smem, st>>>(C, c->T, evals, V, c->status, c->tune[HOLO_TUNE_EIG_MAX_SWEEPS]);
    HOLO_CUDA_OK(cudaGetLastError());
    return HOLO_OK;
}
