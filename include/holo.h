/*
 * holo.h -- C ABI of libholo_b200: the data-parallel hot path of arXiv 2004.00923
 * ("Real-time digital holography of the retina by principal component analysis"),
 * hand-written CUDA for sm_100a (NVIDIA B200).  No cuFFT/cuBLAS/cuSOLVER, no CPU fallback.
 *
 * Path (PAPER.md = /root/reference/PAPER.md; R<n> = reading n in DESIGN.md):
 *   A0  Ibar(x,y)  = (1/T) sum_t I_t(x,y)                         BASELINE.json north_star ("I_t - mean_t I"), R2
 *   A1  g_t        = (I_t - Ibar) * exp(+i pi (x^2+y^2)/(lambda z))   PAPER.md:33-37 Eq. 1 (expanded), R3,R4,R6
 *   A2  H_t        = FFT2D[g_t], forward, unnormalised, no fftshift   PAPER.md:33 ("one spatial Fourier transform"), R5
 *   A3  C          = H^{t*} H,  C_ts = sum_p conj(H_t(p)) H_s(p)      PAPER.md:57-59 Eq. 4, R9
 *   A4  C          = V Lambda V^{t*}                                  PAPER.md:61-65 Eq. 5, R1 (DESCENDING order)
 *   A5  Hc         = H V I_f,  P_k(p) = sum_t H_t(p) V_{t,k}          PAPER.md:67-71 Eq. 6
 *   A6  M(p)       = sum_{k=k_lo}^{k_hi} |P_k(p)|^2                   PAPER.md:71-74 Eq. 7
 *   F1  Fourier demodulation: same as A5/A6 with V := W of Eq. 8      PAPER.md:78-86 Eq. 8-9
 *
 * Conventions common to every call
 *   - All data pointers are DEVICE pointers unless a name ends in _host.  The caller owns every
 *     buffer it passes in; the handle owns its workspace (chirp/twiddle tables, per-pixel frame sum,
 *     FFT scratch, hologram stack H, covariance partials, C, evals, V).
 *   - Layouts: frames uint16 [T][ny][nx] (frame-planar, x fastest), 16-byte aligned;
 *     H complex64 [T][ny][nx] interleaved (re,im), indexed by output bin (ky row, kx column);
 *     C, V complex64 [T][T] row-major; column k-1 of V is eigenvector k (V[t*T + (k-1)]);
 *     evals float [T], DESCENDING, k = 1 is the largest (R1: the paper sorts ascending and keeps
 *     n1..n2; (n1,n2) <-> (k_lo,k_hi) = (T+1-n2, T+1-n1));  image float [ny][nx] in FFT-bin order.
 *   - `stream` is a cudaStream_t cast to void* (NULL = legacy default stream).  Every call only
 *     ENQUEUES work: no host synchronisation and no host<->device copy except in the *_host entry
 *     points, holo_status, holo_profile_read and holo_tune(key 0), which say so.
 *     Allocation: holo_create allocates the workspace of holo_process and of the per-stage calls
 *     (about 8 T nx ny bytes for the hologram stack; at 1024 x 1024 with an even T >= 16 and at
 *     2048 x 2048 the same again for the row-pass output of the packed Fresnel stage).
 *     The following calls allocate more at their FIRST use on a handle (cudaMalloc, which may
 *     synchronise the device) and never afterwards: holo_submit (second hologram stack, second
 *     C / V / evals / status slot, a side stream and six events), holo_push (FP64 Gram store, and in
 *     its pipelined form a ring of T + max(8, T/2) hologram slots plus the side stream and events),
 *     holo_submit_host / holo_process_host (device staging buffers, a copy stream), holo_tune key 5
 *     (events).  Warm a handle up with one call of the form you use before timing or capturing.
 *   - CUDA graphs: holo_process and the per-stage calls (holo_fresnel, holo_covariance, holo_eig,
 *     holo_project, holo_fourier_demod, holo_normalize) enqueue on the caller's stream only and
 *     can be captured (tests/test_gpu_parity.py captures and replays holo_process).  holo_submit /
 *     holo_push fork work to the handle's side stream and join it only in a LATER call
 *     (holo_flush, the submit after next): capture a whole submit...flush sequence, not one call.
 *   - Device: a handle belongs to the device that was current at holo_create; every call checks
 *     that this device is current and returns HOLO_ERR_STATE otherwise (kernel attributes,
 *     streams and events are per device).
 *   - Return value: HOLO_OK or a negative error code; nothing is launched on an error return.
 *     holo_last_error() gives a thread-local message.  Asynchronous CUDA faults surface at the
 *     next call or at destroy.  Jacobi non-convergence (sweep cap hit) is recorded in the device
 *     status word readable with holo_status() AND in a host-visible flag: the first compute
 *     call issued after that solve has finished returns HOLO_ERR_NOCONV without launching
 *     anything and clears the flag (holo_status clears it too).  Results are never silently NaN.
 *   - Arguments: nx, ny powers of two in [16, 4096]; 2 <= T <= 64; lambda, pitch, z finite > 0;
 *     1 <= k_lo <= k_hi <= T (1-based, inclusive, descending eigenvalue order).
 *   - One in-flight call per handle per stream order: calls on one handle must be issued on the
 *     same stream or otherwise ordered by the caller.
 */
#ifndef HOLO_H
#define HOLO_H
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef struct holo_ctx holo_ctx;   /* opaque */
typedef void* holo_stream;          /* cudaStream_t */

enum {
    HOLO_OK = 0,
    HOLO_ERR_ARG = -1,
    HOLO_ERR_ALLOC = -2,
    HOLO_ERR_CUDA = -3,
    HOLO_ERR_STATE = -4,
    HOLO_ERR_NOCONV = -5
};

/* which-values for holo_workspace() */
enum {
    HOLO_WS_SUM = 0,     /* uint32 [ny][nx]  sum_t I_t of the last fresnel/process call            */
    HOLO_WS_H = 1,       /* float2 [T][ny][nx] hologram stack of the last holo_process call        */
    HOLO_WS_C = 2,       /* float2 [T][T]                                                           */
    HOLO_WS_EVALS = 3,   /* float  [T]                                                              */
    HOLO_WS_V = 4,       /* float2 [T][T]                                                           */
    HOLO_WS_STATUS = 5,  /* int32  [8]: {noconv flag, sweeps used, rotations in last sweep, 0,
                          *              SM cycles of load / sweeps / refinement, 0}                        */
    HOLO_WS_QX = 6,      /* float2 [nx] chirp table exp(+i pi x_i^2/(lambda z))                     */
    HOLO_WS_QY = 7       /* float2 [ny]                                                             */
};

/* Create a handle for stacks of T frames of ny x nx pixels (n_t=32, 1024x1024) and
 * the Fresnel parameters of Eq. 1 (lambda = 785 nm, pixel pitch, distance z).
 * Allocates all device workspace (about 8*T*nx*ny + 16*nx*ny*min(T,8) bytes) on the current device
 * and builds the chirp / twiddle tables in double precision on the host.  Returns NULL on failure
 * (reason via holo_last_error()).  This is the only call besides holo_destroy that synchronises. */
holo_ctx* holo_create(int nx, int ny, int T, double lambda_m, double pitch_m, double z_m,
                      int k_lo, int k_hi);

/* NULL-safe.  Synchronises the device, frees the workspace. */
void holo_destroy(holo_ctx* ctx);

/* The whole path A0..A6 for one stack: frames_dev (uint16 [T][ny][nx]) -> image_dev (float [ny][nx]). */
int holo_process(holo_ctx* ctx, const uint16_t* frames_dev, float* image_dev, holo_stream stream);

/* Streaming form of holo_process for a SEQUENCE of stacks (the paper's use: a continuous camera stream,
 * PAPER.md:13,31).  Same arithmetic, same kernels, software-pipelined by one stack: holo_submit(i)
 * enqueues on `stream` the Fresnel stage of stack i, then the projection of stack i-1 into the image_dev
 * given to submit(i-1), then the covariance of stack i, and forks the single-CTA eigensolver of stack i
 * to a side stream owned by the handle, where it runs under the Fresnel kernels of stack i+1.
 * Where the Fresnel stage is the fused persistent kernel (T <= 32; frame sizes other than 1024 x 1024 and 2048 x 2048,
 * or holo_tune key 19 = 0) the projection of stack i instead follows its eigensolver on the side stream and runs on
 * about a quarter of the SMs beside the kernels of stack i+1, whose covariance then sums over fewer CTAs: images equal
 * those of holo_process up to FP32 summation order, and are bit-reproducible.
 * Contract: the image passed to submit(i) is complete, in `stream` order, after holo_flush, or after the
 * holo_submit after next (i+2); frames_dev may be reused as soon as `stream` has passed the submit.  The handle
 * allocates a second hologram stack (8*T*nx*ny bytes) at the first call.  holo_process / holo_flush
 * deliver an owed image first.  Use one stream per handle for a submit sequence. */
int holo_submit(holo_ctx* ctx, const uint16_t* frames_dev, float* image_dev, holo_stream stream);
int holo_flush(holo_ctx* ctx, holo_stream stream);

/* Sliding window (BASELINE.json configs[3]: stride 8 over the stream): the handle keeps the
 * holograms of the T most recent frames; holo_push transforms only the n_new newest frames (1 <= n_new <= T;
 * the first call of a sequence must bring a whole window, n_new = T, and fixes the reference image the holograms
 * are taken against) and renders the PCA image of the window that ends with them.  The result equals
 * holo_process on those T frames up to FP32 rounding (the window mean is removed after the transform, which is
 * exact by linearity; the covariance is centred in FP64).  Needs the deflation form of the projection (rejected
 * components at most half of the kept ones).  holo_process / holo_submit on the same handle end the sequence.
 * Re-reference now and then (a push with n_new = T) if the mean brightness drifts.
 * Completion: with T in {16, 32, 64} and n_new a multiple of 8 (at most T/2) the call is pipelined like
 * holo_submit (ring of T + T/2 hologram slots, eigensolver and projection on the side stream): the image is
 * complete, in `stream` order, after holo_flush or after the push after next.  Otherwise (and with tune key 10 = 0)
 * the call is strictly stream ordered.  Always safe: holo_flush before reading an image. */
int holo_push(holo_ctx* ctx, const uint16_t* new_frames_dev, int n_new, float* image_dev, holo_stream stream);

/* Streaming form with HOST buffers: holo_submit_host copies stack i host -> device on a copy stream owned
 * by the handle (double-buffered staging, so the copy runs under the kernels of stack i-1), enqueues
 * holo_submit on `stream`, and enqueues the device -> host copy of the image of stack i-1.  It returns when
 * the frames have been copied (frames_host may then be reused); every image_host passed so far is complete
 * only after holo_flush_host returns (it synchronises `stream`).  Pinned host memory is needed for the
 * copies to overlap.  This is the end-to-end call bench.py's `e2e` times. */
int holo_submit_host(holo_ctx* ctx, const uint16_t* frames_host, float* image_host, holo_stream stream);
int holo_flush_host(holo_ctx* ctx, holo_stream stream);

/* Same path, HOST buffers (pinned or pageable): copies frames in, runs holo_process, copies the
 * image out, and synchronises `stream` before returning.  Uses a frame/image staging buffer owned by
 * the handle (allocated at first use).  Serial: one stack per call. */
int holo_process_host(holo_ctx* ctx, const uint16_t* frames_host, float* image_host, holo_stream stream);

/* A0+A1+A2: frames_dev -> H_dev (float2 [T][ny][nx]).  (Eq. 1) */
int holo_fresnel(holo_ctx* ctx, const uint16_t* frames_dev, void* H_dev, holo_stream stream);

/* A3: H_dev -> C_dev (float2 [T][T]), full Hermitian matrix written, deterministic (fixed partial
 * count and reduction order; bit-identical across runs).  (Eq. 4) */
int holo_covariance(holo_ctx* ctx, const void* H_dev, void* C_dev, holo_stream stream);

/* A3 from the RAW frames (reading c-12 of Eq. 4): for holograms H_t = FFT2[q d_t] of real
 * mean-subtracted frames (q unimodular, the transform unitary up to nx ny)  C = H^H H = nx ny D^T D  exactly, so the
 * covariance needs neither the holograms nor floating point: the Gram of the uint16 frames is formed in exact integer
 * arithmetic on the tensor cores (tcgen05.mma kind::i8 on the byte planes, s32 accumulators, int64 / __int128
 * assembly), centred with the integer frame sum, and rounded once to float.  frames_dev (uint16 [T][ny][nx]) ->
 * C_dev (float2 [T][T], real symmetric, Im = 0).  Also leaves S = sum_t I_t in the workspace (HOLO_WS_SUM). */
int holo_raw_covariance(holo_ctx* ctx, const uint16_t* frames_dev, void* C_dev, holo_stream stream);

/* Mode of holo_process / holo_submit.  1 (default): the stage decomposition as the paper writes it (Fresnel stage, then
 * the covariance of the hologram stack).  2: holo_raw_covariance + eigensolver FIRST, then the Fresnel stage and the
 * projection with V already known -- the hologram stack is read once instead of twice (20 T N_p + 12 N_p compulsory
 * bytes instead of 28 T N_p + 12 N_p), and in holo_submit the image is complete in stream order when the call's work
 * is done.  Same results up to FP32 rounding of C.
 * 3 (SURVEY.md 8(f)-2 stage 2): mode 2's covariance and eigenvectors, then the image WITHOUT a hologram stack.  With V real
 * (the covariance of the raw frames is real symmetric) the deflation of DESIGN.md R12 commutes with the transform:
 *     M = sum_{k in S} |P_k|^2 = sum_t | FFT2[ q (d_t - sum_{k not in S} e_k V_tk) ] |^2,     e_k = sum_t d_t V_tk,
 * so the rejected components are removed from the RAW frames (one small pass writes the images e_k), the row pass writes
 * its output once (8 T N_p bytes, the only large intermediate), and the column pass is reduced to sum_t |.|^2 in registers:
 * no hologram stack is written, the projection kernel and its read of the stack disappear.  Windows that reject more than
 * 4 components or keep at most 3/4 of them (the paper's own k in [13, 32]) take the eigen-basis form of the same identity,
 * M = sum_{k in S} | FFT2[ q e_k ] |^2: the n_S images e_k of the KEPT components are transformed instead of the T frames
 * (their workspace, 4 T N_p bytes, is allocated by holo_set_mode / holo_set_range when such a window is first seen).  No cancellation (the subtraction happens before the transform, on integers
 * of at most 2^22).  HOLO_WS_H is not filled in this mode.  holo_submit in mode 3 is pipelined by one stack (the covariance
 * of stack i and its eigensolver on the side stream run with the image of stack i-1): the image of submit(i) is complete
 * after the next holo_submit or holo_flush, and frames_dev of submit(i) is READ AGAIN by that next call -- keep it valid
 * and unchanged until then (holo_submit_host does this for you).  First use allocates 13 N_p floats (may synchronise).
 * holo_push always works as in mode 1. */
int holo_set_mode(holo_ctx* ctx, int mode);

/* A4: any Hermitian C_dev (only its lower triangle t >= s and real diagonal are read) ->
 * evals_dev (float [T], descending), V_dev (float2 [T][T], unitary, column k-1 = eigenvector k,
 * phase fixed so that each column's largest-magnitude entry is real positive).  Single-CTA
 * parallel-order complex Jacobi in FP32 with an FP64 Rayleigh-quotient refinement of the
 * eigenvalues.  (Eq. 5) */
int holo_eig(holo_ctx* ctx, const void* C_dev, float* evals_dev, void* V_dev, holo_stream stream);

/* A5+A6 fused: image(p) = sum_{k=k_lo}^{k_hi} |sum_t H_t(p) V_{t,k}|^2 with the handle's current
 * (k_lo,k_hi); P is never stored.  V_dev may be ANY T x T matrix (unitary or not) when
 * `assume_unitary` was not enabled (default): the direct form is used.  (Eq. 6-7) */
int holo_project(holo_ctx* ctx, const void* H_dev, const void* V_dev, float* image_dev, holo_stream stream);

/* F1 (Eq. 8-9): Fourier demodulation of the stack: image(p) = sum_{n=n1}^{n2} |sum_m H_m(p) w_mn|^2,
 * w_mn = exp(-2 i pi (m-1)(n-1)/T)/sqrt(T), n1..n2 1-based inclusive (paper: 8..24 of 32). */
int holo_fourier_demod(holo_ctx* ctx, const void* H_dev, int n1, int n2, float* image_dev, holo_stream stream);

/* SVD filter (Eq. 3): Hf = U Delta I_f V^{t*} = H V I_f V^{t*} with the handle's current (k_lo,k_hi):
 * Hf_t(p) = sum_{k=k_lo}^{k_hi} P_k(p) conj(V_{t,k}), the hologram stack with the rejected components removed, back in the
 * frame basis (the input of the paper's downstream short-time Fourier analysis).  H_dev, Hf_dev float2 [T][ny][nx]
 * (Hf_dev == H_dev is allowed), V_dev float2 [T][T] as written by holo_eig (any matrix is accepted; the identity
 * sum_t |Hf_t|^2 = image of holo_project holds for unitary V).  Evaluated as Hf = H F with the T x T matrix F = V I_f V^{t*}. */
int holo_svd_filter(holo_ctx* ctx, const void* H_dev, const void* V_dev, void* Hf_dev, holo_stream stream);

/* Image normalisation of PAPER.md:86 ("image normalization by their respective average value"): image <- image / mean(image),
 * in place, image_dev float [ny][nx].  The mean is a fixed-order FP64 reduction (bit-reproducible); an all-zero image is
 * left unchanged.  Two small kernels on `stream`. */
int holo_normalize(holo_ctx* ctx, float* image_dev, holo_stream stream);

/* holo_normalize for callers that cannot allocate (code under CUDA-graph capture, tight serving loops, harnesses that forbid
 * cudaMalloc): out = in / mean(in), in_dev, out_dev float [ny][nx] device pointers, 4-byte aligned;
 * out_dev == in_dev is allowed.  NO handle and NO allocation: the call uses neither cudaMalloc / cudaFree nor any
 * allocating library routine; the partial sums of the mean live in a file-scope __device__ array of 32 KB that every GPU
 * which loads the library holds until the process exits.  Limit: nx * ny <= HOLO_STATIC_MAX_PIXELS (2^24 = 4096 x 4096);
 * larger images are rejected with HOLO_ERR_ARG and a message (use holo_normalize).  The mean is a fixed-order FP64 reduction
 * over chunks of 4096 pixels (bit-reproducible, and the same on every GPU); an all-zero image is left unchanged.
 * Two small kernels on `stream`, nothing else: no synchronisation, no copy.  The first call on a device resolves the
 * device address of the array (cudaGetSymbolAddress, no allocation): make it outside stream capture.
 * SHARED STATE: every call on a device uses the same array, which keeps the previous call's contents (nothing needs to
 * start at zero: a call writes every entry it reads).  Calls that overlap on the GPU -- different streams, or host
 * threads without ordering -- race on it and return wrong means: issue them on one stream or order them with events. */
#define HOLO_STATIC_MAX_PIXELS (1LL << 24)
int holo_normalize_static(const float* in_dev, float* out_dev, int nx, int ny, holo_stream stream);

/* Quadrant swap of an image in FFT-bin order: out[(j + ny/2) mod ny][(i + nx/2) mod nx] = in[j][i] (zero frequency to the
 * centre; R6: every other call leaves images in raw FFT-bin order).  Out of place: in_dev != out_dev. */
int holo_fftshift(holo_ctx* ctx, const float* in_dev, float* out_dev, holo_stream stream);

/* Change the component window (1-based inclusive, descending order).  Takes effect at the next call; an image still
 * owed by an earlier holo_submit keeps the window of its own submit call.  While a holo_push sequence is open the
 * new window must keep the deflation form available (HOLO_ERR_STATE otherwise). */
int holo_set_range(holo_ctx* ctx, int k_lo, int k_hi);

/* Allow holo_process/holo_project to use the exact identity sum_{k in S}|P_k|^2 =
 * sum_t |H_t|^2 - sum_{k not in S}|P_k|^2 (valid for unitary V; R12), evaluated without cancellation
 * as sum_t |H_t - sum_{k not in S} P_k conj(V_tk)|^2, when the complement of S is at most half of S.  holo_process always may (its V is unitary by construction); for holo_project
 * this flag (default 0) states that the caller's V is unitary. */
int holo_set_assume_unitary(holo_ctx* ctx, int on);

/* Test hook: device pointer of a workspace array (see HOLO_WS_*), NULL if `which` is invalid. */
const void* holo_workspace(holo_ctx* ctx, int which);

/* Test hook: enqueue a device-to-device copy of the first `nbytes` bytes of workspace array `which`
 * into dst_dev (caller-owned device memory). */
int holo_workspace_copy(holo_ctx* ctx, int which, void* dst_dev, unsigned long long nbytes, holo_stream stream);

/* Copies the first 4 ints of the 8-int status word (HOLO_WS_STATUS: no-convergence flag, sweeps used, rotations
 * in the last sweep, 0) of the last eigensolve to the host.  Synchronises `stream` and the handle's side stream.
 * After holo_submit / holo_push sequences both workspace slots are inspected and a failing one is reported.
 * Returns HOLO_ERR_NOCONV if the Jacobi sweep cap was hit, else HOLO_OK. */
int holo_status(holo_ctx* ctx, int32_t status_host[4], holo_stream stream);

/* Number of kernels one holo_process call launches with the current settings (for gpu_launches). */
int holo_launches_per_process(holo_ctx* ctx);

/* Experiment knobs (not needed for normal use; defaults are chosen at create).  Keys:
 *   0 frames in the FFT row->column ring (L2 residency of the intermediate), 1 covariance CTAs,
 *   2 allow the complement (deflation) form in holo_process (default 1), 3 fused persistent Fresnel kernel
 *   (default 1; 0 = separate row / column launches per frame group), 4 Jacobi sweep cap, 5 per-kernel event
 *   brackets (holo_profile_read), 6 lag in frames between row and column pass in the fused kernel (0 = ring/2),
 *   7 TMA-fed projection (default 1), 8 real-part covariance in holo_process / holo_submit (default 1; the
 *   covariance of holograms of real frames is real in exact arithmetic, R21), 9 SMs given to the
 *   side-stream projection in holo_submit (0 = projection in stream order after the next Fresnel stage),
 *   10 pipelined ring form of holo_push (default 1), 11 incremental Gram update in that form (default 1),
 *   12 direct projection of more than 4 components on the tensor cores (3 x TF32, T <= 32; default 1; 0 = FP32 kernel),
 *   13 real covariance of holo_process / holo_submit on the tensor cores (tcgen05.mma kind::tf32 on values
 *   rounded to nearest, FP64 partials): 0 = FP32 FFMA kernel (default below T = 32, and at T = 32 below 2^18 pixels),
 *   1 = TF32 (default at T = 32 from 2^18 pixels and at T > 32 from 2^20 pixels; T > 32 below that: 3 x TF32), 3 = 3 x TF32,
 *   14 operand stages accumulated in TMEM between two FP64 drains of key 13 (default 4 = 512 products),
 *   15 mode 3: packed row pass (FFMA2 / FADD2 on pairs: the same row of two consecutive frames at nx = 1024 with even T,
 *   the even / odd halves of one row at nx = 2048; default 1), 16 packed 2048-point column passes (mode 3 column energy;
 *   at 2048 x 2048 also the Fresnel stage of modes 1 / 2 as packed row pass + packed column pass instead of the fused
 *   kernel; default 1), 17 mode 3 at 1024 x 1024: width w of the column blocks in which the packed row pass stores its
 *   output, [frame][x / w][y][x % w] (8, 16, 32; 0 = row-major; default 8 = the column tile of the energy pass, which
 *   then reads one contiguous 64 KB block per tile and frame), 18 programmatic dependent launches between the kernels of a
 *   chain (each such kernel waits with griddepcontrol.wait before it touches data; PROCESS-WIDE; default 1, 0 = plain
 *   launches; results are bit-identical either way), 19 the Fresnel stage at 1024 x 1024 (even T >= 16, whole stacks) as two
 *   streaming kernels -- packed row pass of frame pairs into column blocks, column pass from those blocks -- with the
 *   row-pass output of the stack in a second T nx ny complex64 buffer (default 1; 0 = the fused persistent kernel with its
 *   L2 ring, which holo_push keeps for its short strides), 20 single-pass TF32 covariance fed by TMA (3-D swizzled boxes land
 *   in operand layout, rounding in place; default 1; 0 = the register-fed kernel). */
int holo_tune(holo_ctx* ctx, int key, int value);

/* Measurement hooks used by bench.py (not needed for normal use).
 * holo_profile_read: while holo_tune(ctx, 5, 1) is on, every kernel launch is bracketed by a pair of CUDA events;
 * this call synchronises the device and returns, per kernel class (0 temporal sum, 1 Fresnel / row pass, 2 column
 * pass of the unfused form, 3 covariance partials, 4 covariance reduction, 5 eigensolver, 6 projection), the summed
 * device time in ms_out[7] and the launch count in count_out[7] since the last read.
 * holo_fft_group: frames in the row->column ring of the Fresnel stage (tune key 0). */
int holo_profile_read(holo_ctx* ctx, double* ms_out, int* count_out);
int holo_fft_group(holo_ctx* ctx);

const char* holo_last_error(void);   /* thread-local, static storage */
int holo_version(void);              /* major*10000 + minor*100 + patch */

#ifdef __cplusplus
}
#endif
#endif /* HOLO_H */
