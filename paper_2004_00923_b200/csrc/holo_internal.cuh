// holo_internal.cuh -- private declarations shared by the translation units of libholo_b200.
// Product code (CUDA, sm_100a).  Nothing here is shared with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>
#include "../../include/holo.h"

#define HOLO_MAX_T 64
#define HOLO_NUM_TUNE 24
#define HOLO_NORM_PARTS 1024

// tuning keys (holo_tune); not part of the stable ABI
enum {
    HOLO_TUNE_FFT_GROUP = 0,     // frames per row/column pass group (scratch = group * 8*nx*ny bytes)
    HOLO_TUNE_COV_GRIDX = 1,     // covariance CTAs along pixels
    HOLO_TUNE_PROJ_COMPLEMENT = 2, // 1 = allow complement form in holo_process (default 1)
    HOLO_TUNE_FFT_PERSISTENT = 3,  // 1 = k_fresnel (single persistent kernel, default), 0 = separate row / column launches
    HOLO_TUNE_EIG_MAX_SWEEPS = 4,
    HOLO_TUNE_PROFILE = 5,         // 1 = bracket every kernel launch with events (holo_profile_read)
    HOLO_TUNE_PROJ_TMA = 7,        // 1 = deflation projection fed by a TMA ring (default), 0 = register-streaming kernel
    HOLO_TUNE_COV_REAL = 8,        // 1 = holo_process / holo_submit compute Re C only (C is real there, R21); default 1
    HOLO_TUNE_SPLIT_SMS = 9,       // holo_submit: k > 0 = projection on the side stream on k SMs, concurrent with the
                                   // next covariance on the other SMs (memory-bound next to ALU-bound); 0 = in stream order
    HOLO_TUNE_PUSH_PIPE = 10,      // holo_push: 1 = pipelined ring form when T in {16,32,64} and n_new is a multiple of 8 (default)
    HOLO_TUNE_PUSH_INCR = 11,      // holo_push (ring form): 1 = recompute only the Gram rows / columns of the new frames (default)
    HOLO_TUNE_COV_TF32 = 13,       // real covariance of holo_process / holo_submit on the tensor cores: 0 = FP32 FFMA kernel,
                                   // 1 = TF32 (inputs rounded to nearest), 3 = 3 x TF32 split; default 1 at T > 32, else 0
    HOLO_TUNE_COV_TF32_DRAIN = 14,
    HOLO_TUNE_PROJ_TC = 12,        // direct projection of more than 4 components on the tensor cores (T <= 32; default 1)
    HOLO_TUNE_ROWS2 = 15,          // mode 3: packed two-frame row pass where supported (1024^2, even T) // stages accumulated in TMEM before the accumulators are added to FP64 (default 4)
    HOLO_TUNE_TILED_G = 17,        // mode 3, 1024 x 1024: the row pass writes its output column tile by column tile (default 1)
    HOLO_TUNE_PACKED1024 = 19,     // 1024 x 1024 Fresnel stage as packed row pass + column pass (default 1; 0 = fused kernel)
    HOLO_TUNE_COV_TF32_TMA = 20,   // single-pass TF32 covariance fed by TMA (swizzled boxes, in-place rounding; default 1; 0 = register-fed kernel)
    HOLO_TUNE_PDL = 18,            // programmatic dependent launches between the kernels of a chain (process-wide; default 1)
    HOLO_TUNE_COLS2048 = 16,       // mode 3: packed column-energy pass for 2048-point columns (default 1)
    HOLO_TUNE_FFT_LAG = 6,         // frames between the row pass and the column pass in the fused kernel (0 = auto)
};

// kernel classes for the profile hook
enum { HOLO_K_SUM = 0, HOLO_K_FFT_ROWS, HOLO_K_FFT_COLS, HOLO_K_COV_PARTIAL, HOLO_K_COV_REDUCE, HOLO_K_EIG, HOLO_K_PROJECT, HOLO_K_COUNT };
#define HOLO_PROF_CAP 4096

struct FftPlan {            // one 1-D FFT length
    int N;                  // length
    int E;                  // elements per thread per pass (16 or 32)
    int R1, R2;             // radices of pass 1 and 2 (1 = absent); pass 0 is radix E
    int tps;                // threads per sequence = N / E
    float2* tw1;            // device: pass-1 twiddles [R1][E]          exp(-2 pi i r k /(E R1))
    float2* tw2;            // device: pass-2 twiddles [R2][E*R1]
};

struct holo_ctx {
    int nx, ny, T;
    long long npix;
    double lambda_m, pitch_m, z_m;
    int k_lo, k_hi;
    int assume_unitary;
    int device, num_sms;
    int tune[HOLO_NUM_TUNE];
    // tables
    float2 *qx, *qy;        // chirp, separable (built in double on the host)
    float2* qxs;            // qx / T (the mean-subtraction scale folded into the row-pass prologue)
    FftPlan px, py;
    float2* Wdft;           // Eq. 8 DFT basis [T][T]
    float2* Fmat;           // [T][T] filter matrix V I_f V^H of holo_svd_filter (Eq. 3)
    double* norm_partials;  // [HOLO_NORM_PARTS] partial sums of holo_normalize
    // workspace
    uint32_t* sum;          // [ny][nx]
    float2* rowout;         // 2048 x 2048 and 1024 x 1024 (even T) frames: row-pass output of the whole stack [T][ny][nx] (unfused packed Fresnel stage)
    float2* scratch;        // FFT row->column intermediate, fft_group frames
    int scratch_frames;
    float2* H;              // [T][ny][nx]
    float2* cov_partials;   // [cov_parts_cap][T8][T8]
    int cov_nparts;         // partials written by the last covariance launch
    int cov_parts_cap;
    float2* C;
    float* evals;
    float2* V;
    float* defl_img;        // mode 3: [4][ny][nx] raw-domain images of the rejected components (allocated at first use)
    float* defl_coef;       // mode 3: [T][4] their eigenvector entries
    float* energy_parts;    // mode 3: [splits][ny][nx] partial energy images
    float* eig_img;         // mode 3, eigen-basis form: [T][ny][nx] raw-domain images of the kept components (allocated when a window needs it)
    uint32_t* sum1;         // mode 3, streaming form: frame sum of the second slot
    const uint16_t* pend3_frames; float* pend3_image; int pend3_slot;   // mode 3, streaming form: the stack whose image is owed
    unsigned long long* gram_X;   // [128][128] int64 byte-plane Gram of the raw frames (mode 2, rawgram.cu)
    int fresnel_sm_reserve;       // SMs the fused Fresnel launch leaves free (set around the launch by mode 2's holo_submit)
    int gram_nparts;              // CTAs of the last k_sum_gram launch
    unsigned long long* gram_Xp;  // [N (N + 1) / 2][3 num_sms] per-CTA partials of it (N = 64 or 128)
    int mode;               // 1: covariance from the hologram stack (Eq. 4 as written); 2: from the raw frames
    int32_t* status;        // [8], see HOLO_WS_STATUS
    int32_t* noconv_host;   // pinned, mapped host word: set by the eigensolver when it hits the sweep cap (device alias below)
    int32_t* noconv_dev;
    unsigned int* counters; // persistent-kernel tickets / dependency counters
    // profile hook
    cudaEvent_t* prof_ev;   // [2*HOLO_PROF_CAP]
    int* prof_cls;
    int prof_n;
    // streaming form (holo_submit / holo_flush): second workspace slot, side stream for the eigensolver
    float2* H1; float2* C1; float* evals1; float2* V1; int32_t* status1;
    cudaStream_t side;
    cudaEvent_t ev_cov[2], ev_eig[2];
    float* pend_image;      // image of the stack whose projection is still owed (nullptr: none)
    int pend_slot, pend_k_lo, pend_k_hi, pend_complement;   // its workspace slot and the component window at submit time
    long long nsubmit;
    cudaEvent_t ev_proj[2]; int proj_recorded[2];
    // sliding-window form (holo_push)
    double2* Cd;            // [T][T] unrounded Gram sums (allocated at the first push)
    int center_gram;        // 1 while a push is being enqueued: the reduction also centres (C = J Gamma J)
    int push_ready, push_head;   // ring = H: slot push_head is the oldest frame
    // pipelined push: a ring of ring_slots > T hologram slots; the current window starts at slot ring_a.  While
    // ring_nrb != 0 the covariance / projection launchers read the window through the ring (8-row blocks modulo).
    float2* ring; int ring_slots, ring_a; long long npush;
    int ring_rb0, ring_nrb;
    double* Gs;             // [ring_slots][ring_slots] slot-indexed FP64 Gram of the ring (incremental update)
    int cov_new_blocks;     // > 0: the next covariance launch recomputes only the products with the newest 8-frame blocks
    int cov_grid_cap, proj_grid_cap;   // CTA caps used by the SM-split mode of holo_submit (0 = none)
    // host staging for holo_process_host
    uint16_t* frames_stage;
    float* image_stage;
    // streaming host entry (holo_submit_host / holo_flush_host): double-buffered staging + copy stream
    uint16_t* fstage[3]; float* istage[2];      // (the third frame stage only in mode 3, whose frames are read again one call later)
    cudaStream_t copy;
    cudaEvent_t ev_h2d[3], ev_free[3];
    float* pend_image_host; int pend_islot;
    float* pend_host_slot[2];          // SM-split mode: host image owed per staging slot
    long long nsubmit_host;
};

void holo_set_error(const char* fmt, ...);
// Programmatic dependent launch: a kernel launched with holo_launch_pdl may be made resident while the kernel before it in
// the stream is still running (after every CTA of that one has called pdl_trigger or exited), which hides its launch
// latency; it must call pdl_wait() before it reads or writes anything another kernel touches (pdl_wait returns when the
// kernels before it are complete and their writes visible; a no-op in a plain launch).
extern int holo_pdl_enabled;      // process-wide (holo_tune key 18): 0 = plain launches everywhere
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_trigger() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
template <class... KArgs, class... Args>
static inline cudaError_t holo_launch_pdl(void (*kern)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, Args... args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at; cfg.numAttrs = holo_pdl_enabled ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, kern, KArgs(args)...);
}

#define HOLO_CUDA_OK(expr)                                                              \
    do {                                                                                \
        cudaError_t _e = (expr);                                                        \
        if (_e != cudaSuccess) {                                                        \
            holo_set_error("%s failed: %s (%s:%d)", #expr, cudaGetErrorString(_e), __FILE__, __LINE__); \
            return HOLO_ERR_CUDA;                                                       \
        }                                                                               \
    } while (0)

// RAII event bracket around one kernel launch (only when profiling is on)
struct HoloProf {
    holo_ctx* c; cudaStream_t st; int slot;
    HoloProf(holo_ctx* c_, int cls, cudaStream_t st_) : c(c_), st(st_), slot(-1) {
        if (c->tune[HOLO_TUNE_PROFILE] && c->prof_ev && c->prof_n < HOLO_PROF_CAP) {
            slot = c->prof_n++;
            c->prof_cls[slot] = cls;
            cudaEventRecord(c->prof_ev[2 * slot], st);
        }
    }
    ~HoloProf() { if (slot >= 0) cudaEventRecord(c->prof_ev[2 * slot + 1], st); }
};

// stage launchers (each only enqueues on `st`)
int holo_launch_sum(holo_ctx* c, const uint16_t* frames, cudaStream_t st);
int holo_launch_fresnel(holo_ctx* c, const uint16_t* frames, float2* H, cudaStream_t st, bool with_sum = true, int nproc = -1,
                        bool counters_zeroed = false);
// C == nullptr: partials only; holo_launch_cov_reduce then finishes (possibly on another stream, ordered after)
int holo_launch_covariance(holo_ctx* c, const float2* H, float2* C, cudaStream_t st, bool real_only = false);
int holo_launch_cov_reduce(holo_ctx* c, int nparts, float2* C, cudaStream_t st);
int holo_launch_cov_tf32(holo_ctx* c, const float2* H, float2* C, cudaStream_t st);   // covtf32.cu
// cudaFuncSetAttribute / occupancy are properties of a (function, device) pair: cached per pair, thread-safe
int holo_ensure_smem_attr(const void* func, int device, size_t bytes);
int holo_cached_occupancy(const void* func, int device, int threads, size_t smem, int* blocks_per_sm);
// real_symmetric: the caller guarantees Im C = 0 (stored so): real rotations, real eigenvectors (Im V = 0 exactly)
int holo_launch_eig(holo_ctx* c, const float2* C, float* evals, float2* V, cudaStream_t st, bool real_symmetric = false);
// mode 0: direct over columns [k_lo,k_hi] of V; mode 1: complement (total - columns outside)
int holo_launch_project(holo_ctx* c, const float2* H, const float2* V, int k_lo, int k_hi,
                        int allow_complement, float* image, cudaStream_t st, int center = 0);
// project_tc.cu: direct projection of wide component windows on the tensor cores (3 x TF32), T <= 32
bool holo_project_tc_supported(const holo_ctx* c, int nS);
int holo_launch_project_tc(holo_ctx* c, const float2* H, const float2* V, int k_lo, int k_hi, float* image, cudaStream_t st);
int holo_fresnel_launch_count(holo_ctx* c);
// mode 3: image = sum_t |FFT2[q (d_t - sum_{k rejected} e_k V_tk)]|^2 without storing the hologram stack (c->sum and V must be ready)
int holo_launch_energy_image(holo_ctx* c, const uint16_t* frames, const float2* V, int k_lo, int k_hi, float* image, cudaStream_t st);
int holo_mode3_splits(const holo_ctx* c, int nframes);
bool holo_mode3_eigen_form(const holo_ctx* c, int k_lo, int k_hi);
// display.cu: PAPER.md:86 normalisation, quadrant swap, Eq. 3 SVD filter
int holo_launch_normalize(holo_ctx* c, float* image, cudaStream_t st);
int holo_launch_fftshift(holo_ctx* c, const float* in, float* out, cudaStream_t st);
int holo_launch_svd_filter(holo_ctx* c, const float2* H, const float2* V, int k_lo, int k_hi, float2* Hf, cudaStream_t st);
// mode 2: S = sum_t I_t and C = nx ny D^T D from the raw frames (tcgen05 int8 Gram, rawgram.cu)
int holo_launch_sum_gram(holo_ctx* c, const uint16_t* frames, float2* C, cudaStream_t st, bool finish = true);
int holo_launch_gram_finish(holo_ctx* c, float2* C, cudaStream_t st);
// packed two-frame row pass of mode 3 (fresnel2.cu): 1024 x 1024 frames, even T
bool holo_rows2_supported(const holo_ctx* c);
bool holo_cols2048_supported(const holo_ctx* c);
int holo_launch_cols2048(holo_ctx* c, const float2* G, float* out, int nframes, int nsplit, cudaStream_t st);
int holo_launch_cols2048_store(holo_ctx* c, const float2* G, float2* H, int nframes, cudaStream_t st);
bool holo_fresnel_is_packed(const holo_ctx* c);      // Fresnel stage of whole stacks = packed row pass + column pass (not the fused kernel)
int holo_launch_rows2(holo_ctx* c, const uint16_t* frames, float2* out, int ndefl, cudaStream_t st, int nframes = 0, int tile_w = 0);
int holo_fft_plan_init(FftPlan* p, int N);
void holo_fft_plan_free(FftPlan* p);
