// spec.cu — host side of the C-ABI library declared in include/spec.h: plan, state machine
// (filter history, accumulation windows, output ring) and kernel launches.  No torch, no CPU
// fallback: every step of the path runs in the kernels of engine.cuh.
#include "../../include/spec.h"

#include <cuda_fp16.h>
#include <cuda_runtime.h>
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>
#include <time.h>

#include <mutex>
#include <type_traits>
#include <vector>

#include "engine.cuh"
#include "passa_pfb.cuh"
#include "fused.cuh"
#include "fused2.cuh"

using namespace spk;

// ------------------------------------------------------------------ errors
static thread_local char g_err[512] = "";
static int fail_cuda(cudaError_t e, const char* what) {
    snprintf(g_err, sizeof(g_err), "%s: %s", what, cudaGetErrorString(e));
    return (e == cudaErrorMemoryAllocation) ? SPEC_ERR_NOMEM : SPEC_ERR_CUDA;
}
#define CK(call)                                            \
    do {                                                    \
        cudaError_t e__ = (call);                           \
        if (e__ != cudaSuccess) return fail_cuda(e__, #call); \
    } while (0)

extern "C" const char* spec_last_error(void) { return g_err; }
extern "C" const char* spec_strerror(int code) {
    switch (code) {
        case SPEC_OK: return "ok";
        case SPEC_ERR_ARG: return "bad argument";
        case SPEC_ERR_STATE: return "call not valid in this state";
        case SPEC_ERR_SIZE: return "wrong size (count, or nsamples not a multiple of nchan)";
        case SPEC_ERR_OVERRUN: return "output ring overrun: read completed accumulations first";
        case SPEC_ERR_CUDA: return "CUDA error";
        case SPEC_ERR_NOMEM: return "out of memory";
        default: return code > 0 ? "ok" : "unknown error";
    }
}

#ifdef SPEC_TUNING
// Tuning builds only (-DSPEC_TUNING, never the default build): plan parameters overridden from the environment.
static int tuning_int(const char* name, int dflt, int lo, int hi) {
    if (const char* e = getenv(name)) { const long v = atol(e); if (v >= lo && v <= hi) return (int)v; }
    return dflt;
}
#endif

// ------------------------------------------------------------------ handle
struct spec_ctx {
    int N, T, P, S, mode, window;
    long M;
    int N1, N2;            // four-step split, N1 == 1 for the single-kernel path
    int numSM;
    bool use_coef;         // FFT mode: multiply by a window?
    float* d_coef = nullptr;     // T*N (PFB) or N (FFT)
    float2* d_twN = nullptr;     // W_N^e (four-step outer twiddle), N entries, only if N1 > 1
    float2* d_twT = nullptr;     // fused path with N1 > 16: twT[p1*N2 + n2] = W_N^{n2 k1(p1)}
    void* d_tcB = nullptr;       // tensor-core first stage (spec_set_option): split fp16 DFT matrix
    bool tc_stage = false;
    bool r2_single = false;      // direct FFT, N = 8192: one k_engine launch, 2 x 4096 via FrontRawR2
    float2* d_tw1 = nullptr;     // W_N1^e (pass A engine), N1 entries
    float2* d_tw2 = nullptr;     // W_N2^e (single / pass B engine), N2 entries
    int* d_perm = nullptr;       // position -> natural channel
    uint8_t* d_hist[3] = {nullptr, nullptr, nullptr};   // three buffers rotate: overlapping launches never write what another reads
    int cur = 0, nhist = 0;
    float4* d_Z = nullptr;       // four-step intermediate, zbatch spectra (fused path: the Z ring)
    float4* d_Y = nullptr;       // FIR output of a batch (two-launch path with N1 > 16, 8 taps)
    int zbatch = 0;
    // fused persistent four-step kernel (fused.cuh)
    bool fused = false;
    int fgrid = 0, fGS = 0, fRING = 0, fna = 2;   // grid, spectra per group, ring groups, producer CTAs per SM
    unsigned* h_err = nullptr;     // mapped pinned word the fused kernel raises when one of its waits times out
    unsigned* d_err = nullptr;
    unsigned* d_flags = nullptr;   // two sets (alternating launches) of: role words, a_done[fcap], b_done[fcap]
    int fcap = 0;
    int fpdl = 1;                  // fused launches use programmatic stream serialisation
    int fpar = 0;                  // which set of counters / which Z ring the next fused launch uses
    const uint8_t* carry_src = nullptr;   // history carry the next fused launch performs itself (see spec_process)
    uint8_t* carry_dst = nullptr;
    size_t carry_bytes = 0;
    unsigned* d_carry_cnt = nullptr;   // device counter the carrying launches signal (fused.cuh)
    unsigned carry_cum = 0;            // its value once every carrying launch queued so far has signalled
    bool hist_by_kernel = false;       // the current history buffer was written by the previous launch's carry
    bool failed = false;               // a CUDA call failed part-way through spec_process: only spec_reset / spec_destroy are valid
    float* dump = nullptr;             // spec_debug_fir: the launch in flight is a DUMP instantiation writing here
    // eight-sub-band modes (spec_create_subbands): a parent handle owns one child handle per sub-band and the
    // buffer the interleaved input is split into; every field above belongs to the children then
    int nsub = 1;
    std::vector<spec_ctx*> subs;
    uint8_t* d_deint = nullptr;
    size_t deint_cap = 0;              // time samples per sub-band the buffer holds
    // CUDA-graph capture of a periodic call sequence (spec_capture_begin / _end / spec_replayed)
    bool capturing = false;
    int cap_cur = 0, cap_fpar = 0, cap_nhist = 0;
    long long cap_count = 0, cap_win_read = 0;
    long long cap_dcount = 0, cap_dwin = 0;   // what one replay of the captured segment advances
    float* d_ring = nullptr;     // nring accumulators of S*N floats, position order, [pos][S]
    int nring = 0;
    float* d_stage = nullptr;    // planar read-out staging, S*N
    long long count = 0;         // spectra since start/reset
    long long win_read = 0;      // completed windows already read
    // streaming helper
    uint8_t* d_sbuf[2] = {nullptr, nullptr};
    size_t sbuf_bytes = 0;
    cudaStream_t side = nullptr;
    cudaEvent_t ev_copied[2] = {nullptr, nullptr}, ev_used[2] = {nullptr, nullptr};
    std::vector<float> h_coef;
    // optional per-kernel timing (spec_profile): class 0 single, 1 pass A, 2 pass B, 3 read-out
    bool prof = false;
    struct Rec { int cls; cudaEvent_t a, b; };
    std::vector<Rec> recs;
    std::vector<cudaEvent_t> pool;
    double prof_ms[4] = {0, 0, 0, 0};
    long prof_n[4] = {0, 0, 0, 0};
};

static void prof_fold(spec_ctx* s) {
    for (auto& r : s->recs) {
        float ms = 0.f;
        if (cudaEventSynchronize(r.b) == cudaSuccess && cudaEventElapsedTime(&ms, r.a, r.b) == cudaSuccess)
            s->prof_ms[r.cls] += ms;
        s->pool.push_back(r.a);
        s->pool.push_back(r.b);
    }
    s->recs.clear();
}
static cudaEvent_t prof_event(spec_ctx* s) {
    cudaEvent_t e = nullptr;
    if (!s->pool.empty()) { e = s->pool.back(); s->pool.pop_back(); }
    else cudaEventCreate(&e);
    return e;
}
struct ProfScope {
    spec_ctx* s; cudaStream_t st; cudaEvent_t a = nullptr, b = nullptr; int cls;
    ProfScope(spec_ctx* s_, int cls_, cudaStream_t st_) : s(s_), st(st_), cls(cls_) {
        s->prof_n[cls]++;
        if (!s->prof) return;
        if (s->recs.size() >= 2048) prof_fold(s);
        a = prof_event(s); b = prof_event(s);
        cudaEventRecord(a, st);
    }
    ~ProfScope() {
        if (!a) return;
        cudaEventRecord(b, st);
        s->recs.push_back({cls, a, b});
    }
};

static size_t block_bytes(const spec_ctx* s) { return (size_t)s->N * 2 * s->P; }
static size_t acc_floats(const spec_ctx* s) { return (size_t)s->S * s->N; }
static long long windows_done(const spec_ctx* s) { return s->count / s->M; }

// radices of the engine for length L
static void radices(int L, int r[3]) {
    switch (L) {
        case 16: r[0] = 16; r[1] = 1; r[2] = 1; break;
        case 32: r[0] = 2; r[1] = 16; r[2] = 1; break;
        case 64: r[0] = 4; r[1] = 16; r[2] = 1; break;
        case 128: r[0] = 8; r[1] = 16; r[2] = 1; break;
        case 256: r[0] = 16; r[1] = 16; r[2] = 1; break;
        case 512: r[0] = 2; r[1] = 16; r[2] = 16; break;
        case 1024: r[0] = 4; r[1] = 16; r[2] = 16; break;
        case 2048: r[0] = 8; r[1] = 16; r[2] = 16; break;
        case 4096: r[0] = 16; r[1] = 16; r[2] = 16; break;
        default: r[0] = r[1] = r[2] = 1; break;
    }
}
// engine position p -> frequency k (digit reversal, engine.cuh header)
static int pos_to_freq(int L, int p) {
    if (L == 1) return 0;
    int r[3];
    radices(L, r);
    const int LA = L / r[0], LB = LA / r[1];
    const int qa = p / LA, qb = (p % LA) / LB, qc = p % LB;
    return qa + r[0] * (qb + r[1] * qc);
}

// engine stage twiddles, laid out [q][j] so that adjacent lanes (adjacent j) read adjacent entries:
//   stage a: (q-1)*LA + ja -> W_L^{ja q};  stage b (3-stage plans): (RA-1)*LA + (q-1)*LB + jb -> W_LA^{jb q}
static void make_stage_twiddles(int L, std::vector<float2>& w) {
    int r[3];
    radices(L, r);
    const int LA = L / r[0], LB = LA / r[1];
    w.clear();
    if (r[1] == 1) { w.push_back(make_float2(1.f, 0.f)); return; }
    for (int q = 1; q < r[0]; q++)
        for (int j = 0; j < LA; j++) {
            const double a = -2.0 * M_PI * (double)((long)j * q % L) / (double)L;
            w.push_back(make_float2((float)cos(a), (float)sin(a)));
        }
    if (r[2] == 1) return;
    for (int q = 1; q < r[1]; q++)
        for (int j = 0; j < LB; j++) {
            const double a = -2.0 * M_PI * (double)((long)j * q % LA) / (double)LA;
            w.push_back(make_float2((float)cos(a), (float)sin(a)));
        }
}

static void make_twiddles(int L, std::vector<float2>& w) {
    w.resize(L);
    for (int e = 0; e < L; e++) {
        const double a = -2.0 * M_PI * (double)e / (double)L;
        w[e] = make_float2((float)cos(a), (float)sin(a));
    }
}

// default coefficients (include/spec.h spec_create; reading R1)
static void default_coeffs(const spec_ctx* s, std::vector<float>& h) {
    const int N = s->N;
    if (s->mode == SPEC_MODE_FFT) {
        h.resize(N);
        for (int k = 0; k < N; k++)
            h[k] = (s->window == SPEC_WINDOW_HANN) ? (float)(0.5 - 0.5 * cos(2.0 * M_PI * k / (double)N)) : 1.0f;
        return;
    }
    const long Lh = (long)s->T * N;
    h.resize(Lh);
    for (long k = 0; k < Lh; k++) {
        const double x = ((double)k - 0.5 * (double)Lh) / (double)N;
        const double sinc = (x == 0.0) ? 1.0 : sin(M_PI * x) / (M_PI * x);
        const double w = (s->window == SPEC_WINDOW_HANN) ? 0.5 - 0.5 * cos(2.0 * M_PI * (double)k / (double)Lh) : 1.0;
        h[k] = (float)(sinc * w);
    }
}

// ------------------------------------------------------------------ small kernels
// read-out: position order [pos][S] -> planar natural order [S][N]  (PAPER.md:95 step 6)
// blockIdx.y = which of the accumulations popped by this launch: ring slot (slot0 + y) % nring -> out + y*S*N
__global__ void k_unpermute(float* __restrict__ ring, const int* __restrict__ perm, float* __restrict__ dst,
                            int N, int S, int slot0, int nring) {
    const int a = blockIdx.x * blockDim.x + threadIdx.x;
    if (a >= N) return;
    const int k = perm[a];
    float* __restrict__ acc = ring + (size_t)((slot0 + blockIdx.y) % nring) * S * N;
    float* __restrict__ out = dst + (size_t)blockIdx.y * S * N;
    if (S == 4) {
        const float4 v = ((const float4*)acc)[a];
        ((float4*)acc)[a] = make_float4(0.f, 0.f, 0.f, 0.f);   // read and clear: a free ring slot is always zero
        out[k] = v.x;
        out[(size_t)N + k] = v.y;
        out[(size_t)2 * N + k] = v.z;
        out[(size_t)3 * N + k] = v.w;
    } else {
        out[k] = acc[a];
        acc[a] = 0.f;
    }
}

// test hook: the unpack the kernels use, word by word.  npol = 2: unpack_cpx<2> (the packed form every dual-pol
// front end calls), npol = 1: unpack_cpx<1>
__global__ void k_debug_unpack(const uint8_t* __restrict__ b, size_t n, float* __restrict__ out, int npol) {
    const size_t i = ((size_t)blockIdx.x * blockDim.x + threadIdx.x) * 4;
    if (i >= n) return;
    uint32_t w = 0;
    for (int j = 0; j < 4 && i + j < n; j++) w |= (uint32_t)b[i + j] << (8 * j);
    float f[4];
    if (npol == 2) {
        const float4 z = cpx_to_f4(unpack_cpx<2>(w));   // (Xre, Yre, Xim, Yim)
        f[0] = z.x; f[1] = z.z; f[2] = z.y; f[3] = z.w;
    } else {
        const float4 z0 = cpx_to_f4(unpack_cpx<1>(w & 0xffffu)), z1 = cpx_to_f4(unpack_cpx<1>(w >> 16));
        f[0] = z0.x; f[1] = z0.z; f[2] = z1.x; f[3] = z1.z;
    }
    for (int j = 0; j < 4 && i + j < n; j++) out[i + j] = f[j];
}

// test hook: float4 (Xre, Yre, Xim, Yim) / float2-in-float4 intermediates -> the caller's [n][re,im per pol]
__global__ void k_debug_reorder(const float4* __restrict__ y, size_t n, float* __restrict__ out, int npol) {
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const float4 z = y[i];
    if (npol == 2) ((float4*)out)[i] = make_float4(z.x, z.z, z.y, z.w);
    else ((float2*)out)[i] = make_float2(z.x, z.z);
}

// eight-sub-band modes: the input carries nsub sub-bands interleaved per time sample
// (reading R26): in[j][s] (one word of 2*npol bytes each) -> out[s][j], sub-band s contiguous.
// One thread per time sample: it reads its nsub adjacent words and writes one word to each sub-band's stream,
// so a warp reads 32*nsub contiguous words and writes 32 contiguous words per stream.
template <class W>
__global__ void k_deinterleave(const W* __restrict__ in, W* __restrict__ out, size_t ns, int nsub, size_t out_stride) {
    const size_t j = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= ns) return;
    const W* src = in + j * nsub;
    for (int s = 0; s < nsub; s++) out[(size_t)s * out_stride + j] = __ldg(src + s);
}

// test hook (soak test): one CTA per SM that holds `smem` bytes of shared memory and spins for `ns` nanoseconds
__global__ void __launch_bounds__(128, 1) k_debug_hog(unsigned long long ns, unsigned* sink) {
    extern __shared__ unsigned hog[];
    hog[threadIdx.x] = threadIdx.x;
    unsigned long long t0, t1;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t0));
    do {
        __nanosleep(1000);
        asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t1));
    } while (t1 - t0 < ns);
    if (hog[(threadIdx.x + 1) & 127] == 0xffffffffu) *sink = 1u;
}

// FP32 peak: 16 independent FFMA chains per thread, operands shared so the register file is not
// the limit
__global__ void __launch_bounds__(1024, 1) k_fp32_peak(float* out, int iters, float c0, float c1) {
    float a[16];
#pragma unroll
    for (int i = 0; i < 16; i++) a[i] = (float)(threadIdx.x + i) * 1e-9f;
    for (int it = 0; it < iters; it++) {
#pragma unroll
        for (int i = 0; i < 16; i++) a[i] = fmaf(a[i], c0, c1);
    }
    float sum = 0.f;
#pragma unroll
    for (int i = 0; i < 16; i++) sum += a[i];
    out[blockIdx.x * blockDim.x + threadIdx.x] = sum;
}

// Throughput probes (spec_debug_probe): thread-instructions per clock and SM of the instruction kinds the kernels are
// built from, measured with 8-16 independent chains per thread on every SM.  DESIGN.md section 6 quotes them.
template <int OP>
__global__ void __launch_bounds__(1024, 1) k_probe(float* out, int iters, float c0, float c1) {
    extern __shared__ float4 psm[];
    u64 a[8];
#pragma unroll
    for (int i = 0; i < 8; i++) a[i] = pk(threadIdx.x * 1e-9f + i, (float)i);
    const u64 b = pk(c0 + threadIdx.x * 1e-12f, c0), c = pk(c1, c1);
    float acc = 0.f;
    if (OP >= 4 && OP <= 5) {
        for (int i = threadIdx.x; i < 4096; i += blockDim.x) psm[i] = make_float4((float)i, 1.f, 2.f, 3.f);
        __syncthreads();
    }
    int idx = threadIdx.x;
    for (int it = 0; it < iters; it++) {
        if (OP == 0) {          // scalar FFMA, three register operands (16 per iteration)
#pragma unroll
            for (int i = 0; i < 8; i++) {
                float lo, hi;
                upk(a[i], lo, hi);
                asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(lo) : "f"(c0), "f"(c1));
                asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(hi) : "f"(c0), "f"(c1));
                a[i] = pk(lo, hi);
            }
        } else if (OP == 1) {   // FFMA2 (8)
#pragma unroll
            for (int i = 0; i < 8; i++) asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(a[i]) : "l"(b), "l"(c));
        } else if (OP == 2) {   // FADD2, two distinct register pairs (8)
#pragma unroll
            for (int i = 0; i < 8; i++) asm volatile("add.rn.f32x2 %0, %1, %2;" : "=l"(a[i]) : "l"(a[i]), "l"(a[(i + 3) & 7]));
        } else if (OP == 3) {   // PRMT (16)
#pragma unroll
            for (int i = 0; i < 8; i++) {
                unsigned lo = (unsigned)a[i], hi = (unsigned)(a[i] >> 32);
                asm volatile("prmt.b32 %0, %0, %1, 0x7440;" : "+r"(lo) : "r"((unsigned)b));
                asm volatile("prmt.b32 %0, %0, %1, 0x7440;" : "+r"(hi) : "r"((unsigned)b));
                a[i] = ((u64)hi << 32) | lo;
            }
        } else if (OP == 4 || OP == 5) {   // LDS.128 (4), alone or with 8 FFMA2 behind each
#pragma unroll
            for (int j = 0; j < 4; j++) {
                const float4 v = psm[(idx + j * 1024) & 4095];
                acc += v.x;
                if (OP == 5) {
#pragma unroll
                    for (int i = 0; i < 8; i++) asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(a[i]) : "l"(b), "l"(c));
                }
            }
            idx += 32;
        } else {                // SHFL: one dual-pol point (four words) to another lane (16 shuffles = 4 points)
#pragma unroll
            for (int i = 0; i < 8; i++) {
                unsigned lo = (unsigned)a[i], hi = (unsigned)(a[i] >> 32);
                lo = __shfl_xor_sync(0xffffffffu, lo, 1 + (i & 15));
                hi = __shfl_xor_sync(0xffffffffu, hi, 1 + (i & 15));
                a[i] = ((u64)hi << 32) | lo;
            }
        }
    }
#pragma unroll
    for (int i = 0; i < 8; i++) { float lo, hi; upk(a[i], lo, hi); acc += lo + hi; }
    out[blockIdx.x * blockDim.x + threadIdx.x] = acc;
}

// ------------------------------------------------------------------ launches
template <class K>
static int prep_smem(K kern, size_t bytes) {
    // once per kernel and size (the attributes are sticky; nothing is set again inside a graph capture)
    static std::mutex mu;
    static std::vector<std::pair<const void*, size_t>> done;
    std::lock_guard<std::mutex> lk(mu);
    for (auto& d : done)
        if (d.first == (const void*)kern && d.second >= bytes) return 0;
    done.push_back({(const void*)kern, bytes});
    if (bytes > 48 * 1024) CK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes));
    // ask for the largest shared-memory carve-out: the default heuristic sized it for one or two CTAs
    // per SM and capped the occupancy of these kernels below their register limit
    if (bytes > 0) CK(cudaFuncSetAttribute(kern, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared));
    return 0;
}
static inline int cdiv(long long a, long long b) { return (int)((a + b - 1) / b); }

// Stokes sink of the accumulating kernels: dual-pol transforms of at least 512 points (one warp or
// more per FFT slot) keep their accumulators in tensor memory, everything else in registers
template <class PL, int P>
struct StokesSinkOf {
    static constexpr bool kTmem = (P == 2 && PL::NTS >= 32);
    typedef typename std::conditional<kTmem, SinkStokesTmem, SinkStokes<P>>::type type;
};
static int blocks_by_smem(size_t smem, int cap) {
    const int b = (int)((227 * 1024) / (smem + 1024));
    return b < 1 ? 1 : (b > cap ? cap : b);
}

// accumulating single-kernel launches: consecutive ones may overlap (programmatic stream serialisation, engine.cuh)
template <class K, class... Args>
static cudaError_t launch_pdl(K kern, dim3 grid, int nt, size_t smem, cudaStream_t st, const spec_ctx* s, Args... args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid; cfg.blockDim = dim3(nt); cfg.dynamicSmemBytes = smem; cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at;
    int pdl = s->capturing ? 0 : 1;
#ifdef SPEC_TUNING
    pdl = tuning_int("SPEC_SINGLE_PDL", pdl, 0, 1);
#endif
    cfg.numAttrs = pdl;
    return cudaLaunchKernelEx(&cfg, kern, args...);
}

template <class PL, int MODE_PFB, int P, int WIN>
static int launch_single_w(spec_ctx* s, const InputView& view, long long m0, long long nspec, long long c0,
                           cudaStream_t st) {
    typedef typename StokesSinkOf<PL, P>::type Sink;
    constexpr bool TM = Sink::kTmem;
    constexpr int G = (PL::NTS >= 128) ? 1 : 128 / PL::NTS;
    constexpr int NT = PL::NTS * G;
    // register budget: 128 per thread with TMEM accumulators (512 threads per SM), 168 without
    constexpr int MINB = TM ? 512 / NT : ((NT <= 128) ? 3 : 1);
    const size_t smem = (PL::NST > 1) ? (size_t)G * PL::L * (sizeof(float4) + (MODE_PFB ? 0 : 2 * P)) + 16 : 0;
    FrontRaw<MODE_PFB, P, WIN> front{view, s->d_coef, s->N, s->T, 1, m0};
    Sink sink{s->d_ring, acc_floats(s), s->nring, PL::L, 0};
    const int resident = blocks_by_smem(smem, MINB);
    // one wave: exactly the CTAs the GPU holds at once, each with the longest possible run (the per-CTA prologue --
    // tensor-memory allocation, twiddles, pipeline fill -- is paid once per run), and the next call's launch fills the
    // slots as they free (programmatic dependent launch).  Measured against two waves at 64 MiB calls
    // (profiles/r02_experiments.md): FFT 1024 / 2048 / 4096: 232 -> 298, 291 -> 320, 256 -> 282 GHz
    int waves = 1;
#ifdef SPEC_TUNING
    waves = tuning_int("SPEC_SINGLE_WAVES", 1, 1, 8);
#endif
    const long long target = (long long)s->numSM * resident * waves * G;
    const int len = cdiv(nspec, target);
    const int nruns = cdiv(nspec, len);
    JobMap jm{nspec, len, nruns, 1, nruns, c0, s->M, 1};
    if (s->dump) {   // test hook: the same kernel, front end only
        auto kd = k_engine<PL, false, G, MINB, FrontRaw<MODE_PFB, P, WIN>, Sink, true>;
        int rc = prep_smem(kd, smem);
        if (rc) return rc;
        kd<<<dim3(cdiv(nruns, G)), NT, smem, st>>>(front, sink, jm, s->d_tw2, s->dump);
        CK(cudaGetLastError());
        return 0;
    }
    auto kern = k_engine<PL, false, G, MINB, FrontRaw<MODE_PFB, P, WIN>, Sink>;
    int rc = prep_smem(kern, smem);
    if (rc) return rc;
    {
        ProfScope ps(s, 0, st);
        CK(launch_pdl(kern, dim3(cdiv(nruns, G)), NT, smem, st, s, front, sink, jm, (const float2*)s->d_tw2, (float*)nullptr));
    }
    CK(cudaGetLastError());
    return 0;
}
template <class PL, int MODE_PFB, int P>
static int launch_single(spec_ctx* s, const InputView& view, long long m0, long long nspec, long long c0,
                         cudaStream_t st) {
    if (MODE_PFB || s->use_coef) return launch_single_w<PL, MODE_PFB, P, 1>(s, view, m0, nspec, c0, st);
    return launch_single_w<PL, MODE_PFB, P, 0>(s, view, m0, nspec, c0, st);
}

template <class PL, int MODE_PFB, int P, int WIN>
static int launch_passA_w(spec_ctx* s, const InputView& view, long long m0, int nb, cudaStream_t st) {
    constexpr int G = 256 / PL::NTS;
    const size_t smem = (PL::NST > 1) ? (size_t)G * PL::L * sizeof(float4) : 0;
    FrontRaw<MODE_PFB, P, WIN> front{view, s->d_coef, s->N, s->T, s->N2, m0};
    SinkZ sink{s->d_Z, s->d_twN, s->N, s->N2};
    const int gx = s->N2 / G;
    int ny = cdiv((long long)4 * s->numSM, gx);
    if (ny > nb) ny = nb;
    const int len = cdiv(nb, ny);
    ny = cdiv(nb, len);
    JobMap jm{nb, len, s->N2, 0, 1, 0, 1};
    if (s->dump) {   // test hook: the same kernel, front end only
        auto kd = k_engine<PL, true, G, 1, FrontRaw<MODE_PFB, P, WIN>, SinkZ, true>;
        int rc = prep_smem(kd, smem);
        if (rc) return rc;
        kd<<<dim3(gx, ny), PL::NTS * G, smem, st>>>(front, sink, jm, s->d_tw1, s->dump);
        CK(cudaGetLastError());
        return 0;
    }
    auto kern = k_engine<PL, true, G, 1, FrontRaw<MODE_PFB, P, WIN>, SinkZ>;
    int rc = prep_smem(kern, smem);
    if (rc) return rc;
    {
        ProfScope ps(s, 1, st);
        kern<<<dim3(gx, ny), PL::NTS * G, smem, st>>>(front, sink, jm, s->d_tw1, nullptr);
    }
    CK(cudaGetLastError());
    return 0;
}

template <class PL, int MODE_PFB, int P>
static int launch_passA(spec_ctx* s, const InputView& view, long long m0, int nb, cudaStream_t st) {
    if (MODE_PFB || s->use_coef) return launch_passA_w<PL, MODE_PFB, P, 1>(s, view, m0, nb, st);
    return launch_passA_w<PL, MODE_PFB, P, 0>(s, view, m0, nb, st);
}

template <class PL, int P>
static int launch_passB(spec_ctx* s, int nb, long long c0, cudaStream_t st) {
    typedef typename StokesSinkOf<PL, P>::type Sink;
    constexpr int G = (PL::NTS >= 128) ? 1 : 128 / PL::NTS;
    constexpr int NT = PL::NTS * G;
    constexpr int MINB = Sink::kTmem ? 512 / NT : ((NT <= 128) ? 3 : 1);
    const size_t smem = (size_t)G * PL::L * 2 * sizeof(float4) + 16;
    FrontZ front{s->d_Z, s->N, s->N2};
    Sink sink{s->d_ring, acc_floats(s), s->nring, PL::L, 1};
    const int gx = cdiv(s->N1, G);
    int ny = cdiv((long long)4 * s->numSM, gx);
    if (ny > nb) ny = nb;
    const int len = cdiv(nb, ny);
    ny = cdiv(nb, len);
    JobMap jm{nb, len, s->N1, 0, 1, c0, s->M};
    auto kern = k_engine<PL, false, G, MINB, FrontZ, Sink>;
    int rc = prep_smem(kern, smem);
    if (rc) return rc;
    {
        ProfScope ps(s, 2, st);
        kern<<<dim3(gx, ny), NT, smem, st>>>(front, sink, jm, s->d_tw2, nullptr);
    }
    CK(cudaGetLastError());
    return 0;
}

// direct FFT with N = 2 L in ONE k_engine launch: every spectrum is two slots (even / odd channels), FrontRawR2
template <class PL, int WIN>
static int launch_single_r2(spec_ctx* s, const InputView& view, long long nspec, long long c0, cudaStream_t st) {
    typedef SinkStokesTmem Sink;
    constexpr int G = 1, NT = PL::NTS, MINB = 512 / NT;
    const size_t smem = (size_t)PL::L * (sizeof(float4) + 8) + 16;
    FrontRawR2<WIN> front{view, s->d_twN, s->d_coef, s->N, PL::L, 0};
    Sink sink{s->d_ring, acc_floats(s), s->nring, PL::L, 1};
    const int resident = blocks_by_smem(smem, MINB);
    int waves2 = 1;   // one wave of CTAs, as in launch_single_w (FFT 8192: 198 -> 214 GHz against two)
#ifdef SPEC_TUNING
    waves2 = tuning_int("SPEC_R2_WAVES", 1, 1, 8);
#endif
    const long long target = (long long)s->numSM * resident * waves2 / 2;   // runs (each run is two slots, i.e. two CTAs)
    const int len = cdiv(nspec, target < 1 ? 1 : target);
    const int nruns = cdiv(nspec, len);
    JobMap jm{nspec, len, 2 * nruns, 1, nruns, c0, s->M, 1};
    if (s->dump) {
        auto kd = k_engine<PL, false, G, MINB, FrontRawR2<WIN>, Sink, true>;
        int rc = prep_smem(kd, smem);
        if (rc) return rc;
        kd<<<dim3(2 * nruns), NT, smem, st>>>(front, sink, jm, s->d_tw2, s->dump);
        CK(cudaGetLastError());
        return 0;
    }
    auto kern = k_engine<PL, false, G, MINB, FrontRawR2<WIN>, Sink>;
    int rc = prep_smem(kern, smem);
    if (rc) return rc;
    {
        ProfScope ps(s, 0, st);
        CK(launch_pdl(kern, dim3(2 * nruns), NT, smem, st, s, front, sink, jm, (const float2*)s->d_tw2, (float*)nullptr));
    }
    CK(cudaGetLastError());
    return 0;
}

typedef Plan<16, 16, 1, 1> PL16;
typedef Plan<32, 2, 16, 1> PL32;
typedef Plan<64, 4, 16, 1> PL64;
typedef Plan<128, 8, 16, 1> PL128;
typedef Plan<256, 16, 16, 1> PL256;
typedef Plan<512, 2, 16, 16> PL512;
typedef Plan<1024, 4, 16, 16> PL1024;
typedef Plan<2048, 8, 16, 16> PL2048;
typedef Plan<4096, 16, 16, 16> PL4096;

static int run_single(spec_ctx* s, const InputView& v, long long m0, long long nspec, long long c0, cudaStream_t st) {
    switch (s->N) {
#define SINGLE_CASE(LEN, PLX)                                                       \
    case LEN: {                                                                     \
        const bool pfb = (s->mode == SPEC_MODE_PFB);                                \
        if (pfb && s->P == 2) return launch_single<PLX, 1, 2>(s, v, m0, nspec, c0, st); \
        if (pfb && s->P == 1) return launch_single<PLX, 1, 1>(s, v, m0, nspec, c0, st); \
        if (!pfb && s->P == 2) return launch_single<PLX, 0, 2>(s, v, m0, nspec, c0, st); \
        return launch_single<PLX, 0, 1>(s, v, m0, nspec, c0, st);                  \
    }
        SINGLE_CASE(16, PL16)
        SINGLE_CASE(32, PL32)
        SINGLE_CASE(64, PL64)
        SINGLE_CASE(128, PL128)
        SINGLE_CASE(256, PL256)
        SINGLE_CASE(512, PL512)
        SINGLE_CASE(1024, PL1024)
        SINGLE_CASE(2048, PL2048)
        SINGLE_CASE(4096, PL4096)
#undef SINGLE_CASE
    }
    return SPEC_ERR_ARG;
}

template <int P>
static int launch_passA_pfb16(spec_ctx* s, const InputView& view, long long m0, int nb, cudaStream_t st) {
    constexpr int C = 32, R = 8;
    const size_t smem = (size_t)R * 16 * C * sizeof(float4);
    const int gx = s->N2 / C;
    const int nphases = cdiv(nb, R);
    int ny = cdiv((long long)3 * s->numSM, gx);
    if (ny > nphases) ny = nphases;
    const int ppc = cdiv(nphases, ny);
    ny = cdiv(nphases, ppc);
    if (s->dump) {   // test hook: the same kernel, FIR phase only
        auto kd = k_passA_pfb16<P, 8, C, R, true>;
        int rc = prep_smem(kd, smem);
        if (rc) return rc;
        kd<<<dim3(gx, ny), C * R, smem, st>>>(view, s->d_coef, (float4*)s->dump, s->d_twN, s->N, s->N2, m0, nb, ppc);
        CK(cudaGetLastError());
        return 0;
    }
    auto kern = k_passA_pfb16<P, 8, C, R>;
    int rc = prep_smem(kern, smem);
    if (rc) return rc;
    {
        ProfScope ps(s, 1, st);
        kern<<<dim3(gx, ny), C * R, smem, st>>>(view, s->d_coef, s->d_Z, s->d_twN, s->N, s->N2, m0, nb, ppc);
    }
    CK(cudaGetLastError());
    return 0;
}

// N1 > 16 with the paper's 8 taps: stand-alone sliding FIR into Y, then the column FFTs read Y
template <class PL, int P>
static int launch_passA_fir(spec_ctx* s, const InputView& view, long long m0, int nb, cudaStream_t st) {
    constexpr int CH = 32;
    {
        ProfScope ps(s, 1, st);
        k_fir8<P, CH><<<dim3(cdiv(s->N, 256), cdiv(nb, CH)), 256, 0, st>>>(view, s->d_coef, s->d_Y, s->N, m0, nb);
    }
    CK(cudaGetLastError());
    if (s->dump) {   // test hook: the FIR kernel's own output
        const size_t n = (size_t)nb * s->N;
        k_debug_reorder<<<cdiv((long long)n, 256), 256, 0, st>>>(s->d_Y, n, s->dump, P);
        CK(cudaGetLastError());
        return 0;
    }
    constexpr int G = 256 / PL::NTS;
    const size_t smem = (PL::NST > 1) ? (size_t)G * PL::L * sizeof(float4) : 0;
    FrontY front{s->d_Y, s->N, s->N2};
    SinkZ sink{s->d_Z, s->d_twN, s->N, s->N2};
    const int gx = s->N2 / G;
    int ny = cdiv((long long)4 * s->numSM, gx);
    if (ny > nb) ny = nb;
    const int len = cdiv(nb, ny);
    ny = cdiv(nb, len);
    JobMap jm{nb, len, s->N2, 0, 1, 0, 1};
    auto kern = k_engine<PL, true, G, 1, FrontY, SinkZ>;
    int rc = prep_smem(kern, smem);
    if (rc) return rc;
    {
        ProfScope ps(s, 1, st);
        kern<<<dim3(gx, ny), PL::NTS * G, smem, st>>>(front, sink, jm, s->d_tw1, nullptr);
    }
    CK(cudaGetLastError());
    return 0;
}

static int run_passA(spec_ctx* s, const InputView& v, long long m0, int nb, cudaStream_t st) {
    if (s->mode == SPEC_MODE_PFB && s->N1 == 16 && s->T == 8)
        return (s->P == 2) ? launch_passA_pfb16<2>(s, v, m0, nb, st) : launch_passA_pfb16<1>(s, v, m0, nb, st);
    if (s->d_Y) {
        switch (s->N1) {
#define AF_CASE(LEN, PLX) \
    case LEN: return (s->P == 2) ? launch_passA_fir<PLX, 2>(s, v, m0, nb, st) : launch_passA_fir<PLX, 1>(s, v, m0, nb, st);
            AF_CASE(32, PL32)
            AF_CASE(64, PL64)
            AF_CASE(128, PL128)
#undef AF_CASE
        }
    }
    switch (s->N1) {
#define A_CASE(LEN, PLX)                                                        \
    case LEN: {                                                                 \
        const bool pfb = (s->mode == SPEC_MODE_PFB);                            \
        if (pfb && s->P == 2) return launch_passA<PLX, 1, 2>(s, v, m0, nb, st); \
        if (pfb && s->P == 1) return launch_passA<PLX, 1, 1>(s, v, m0, nb, st); \
        if (!pfb && s->P == 2) return launch_passA<PLX, 0, 2>(s, v, m0, nb, st); \
        return launch_passA<PLX, 0, 1>(s, v, m0, nb, st);                       \
    }
        A_CASE(16, PL16)
        A_CASE(32, PL32)
        A_CASE(64, PL64)
        A_CASE(128, PL128)
#undef A_CASE
    }
    return SPEC_ERR_ARG;
}

static int run_passB(spec_ctx* s, int nb, long long c0, cudaStream_t st) {
    switch (s->N2) {
#define B_CASE(LEN, PLX)                                                   \
    case LEN:                                                              \
        return (s->P == 2) ? launch_passB<PLX, 2>(s, nb, c0, st) : launch_passB<PLX, 1>(s, nb, c0, st);
        B_CASE(64, PL64)
        B_CASE(128, PL128)
        B_CASE(256, PL256)
        B_CASE(512, PL512)
        B_CASE(1024, PL1024)
        B_CASE(2048, PL2048)
        B_CASE(4096, PL4096)
#undef B_CASE
    }
    return SPEC_ERR_ARG;
}

// ---- fused persistent four-step kernel (fused.cuh): one launch per call
static const int FUSED_ROLE_WORDS = kFusedRoleWords;
#ifndef FUSED_PER_SM
#define FUSED_PER_SM 4   // resident CTAs of 128 threads per SM (128 registers each)
#endif
// ---- one persistent grid at a time.  A k_fused grid is exactly what the GPU holds at once and its CTAs wait for one
// another, so two such grids must never become resident piecemeal side by side (each would wait for slots the
// other holds).  Consecutive launches on ONE stream are safe (the dependent launch only starts once its
// predecessor is fully resident); launches on DIFFERENT streams (several handles) are chained here in submission
// order with an event, per device.  The chain costs nothing until a second stream shows up: from then on an
// event is recorded after every persistent launch (which also keeps same-stream launches from overlapping).
struct FusedChain {
    std::mutex mu;
    cudaStream_t last = nullptr;
    bool has_last = false, multi = false, ev_valid = false;
    cudaEvent_t ev = nullptr;
};
static FusedChain g_chain[64];
static FusedChain& fused_chain() {
    int dev = 0;
    cudaGetDevice(&dev);
    return g_chain[dev & 63];
}
// call with the chain locked, before the launch on `st`
static int fused_chain_enter(FusedChain& c, cudaStream_t st) {
    cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
    if (cudaStreamIsCapturing(st, &cap) == cudaSuccess && cap != cudaStreamCaptureStatusNone) return 0;   // a graph node: ordered by the graph
    if (!c.multi && c.has_last && c.last != st) {
        CK(cudaDeviceSynchronize());   // once: everything queued before the second stream appeared has finished
        if (!c.ev) CK(cudaEventCreateWithFlags(&c.ev, cudaEventDisableTiming));
        c.multi = true;
        c.ev_valid = false;
    }
    if (c.multi && c.ev_valid && c.last != st) CK(cudaStreamWaitEvent(st, c.ev, 0));
    return 0;
}
static int fused_chain_leave(FusedChain& c, cudaStream_t st) {
    cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
    if (cudaStreamIsCapturing(st, &cap) == cudaSuccess && cap != cudaStreamCaptureStatusNone) return 0;
    if (c.multi) {
        CK(cudaEventRecord(c.ev, st));
        c.ev_valid = true;
    }
    c.last = st;
    c.has_last = true;
    return 0;
}
// spec_destroy / spec_reset have synchronised the device: nothing persistent is in flight any more
static void fused_chain_quiesce() {
    FusedChain& c = fused_chain();
    std::lock_guard<std::mutex> lk(c.mu);
    c.has_last = false;
    c.ev_valid = false;
    c.multi = false;
}

// the per-group counters of the fused kernel: two sets (alternating launches), each FUSED_ROLE_WORDS + 2*cap words
static int fused_alloc_flags(spec_ctx* s, int ngroups) {
    const int cap = (ngroups + ngroups / 2 + 64) & ~3;
    unsigned* f = nullptr;
    CK(cudaMalloc(&f, (size_t)2 * (FUSED_ROLE_WORDS + 2 * cap) * sizeof(unsigned)));
    cudaError_t e = cudaMemset(f, 0, (size_t)2 * (FUSED_ROLE_WORDS + 2 * cap) * sizeof(unsigned));   // the kernel leaves them zero
    if (e != cudaSuccess) { cudaFree(f); return fail_cuda(e, "cudaMemset(flags)"); }
    cudaFree(s->d_flags);   // (the new set exists before the old one goes: a failed allocation leaves the handle intact)
    s->d_flags = f;
    s->fcap = cap;
    return 0;
}

template <class PL, int NT, int MODE_PFB, int PER_SM, int N1 = 16>
static int fused_do(spec_ctx* s, bool query, const InputView& view, long long nspec, long long c0, cudaStream_t st) {
    constexpr bool kTcOk = (MODE_PFB == 0 && N1 == 16 && NT == 128);   // plans that have a tensor-core first stage
    // plans that run as k_fused2 (both roles per CTA, consumer rows prefetched by bulk copy): direct-FFT mode, and PFB mode
    // at N = 131072 and 262144 (the ring misses the L2 there and the prefetch hides DRAM latency; at 524288 the producer's
    // buffers leave no room for two row buffers, at 65536 it measured slower: sweep 104.8 -> 88.6 GHz).  Measured (profiles/r02_experiments.md): FFT 16384 / 32768
    // 136 -> 149 / 146 GHz, PFB 131072 / 262144 71 -> 82 / 58 -> 71 GHz, but PFB 32768 117 -> 108 GHz (the staged rows add a
    // shared-memory pass to a mode whose shared-memory pipe is already half busy with the FIR hand-off)
    constexpr bool kF2 = PL::NST == 3 && Fused2Shape<PL, MODE_PFB, N1>::kFits && (MODE_PFB == 0 || (NT == 256 && N1 > 16));
    auto kern = k_fused<PL, NT, MODE_PFB, PER_SM, false, N1>;
    auto kern_tc = k_fused<PL, NT, MODE_PFB, PER_SM, false, N1, kTcOk>;
    // exchange buffer / FIR hand-off, plus (PFB) the staged raw tile of a producer phase: R+7 blocks of 1 KiB
    // (N1 > 16: the hand-off buffer of 16 points per thread plus the staged tile of ProducerBig)
    typedef ProducerBig<256, PL::L, (N1 > 16 ? N1 : 32), MODE_PFB ? 8 : 1> Big;
    const size_t smem = (N1 > 16) ? Big::SMEM
                                  : (size_t)NT * 16 * sizeof(float4) + (MODE_PFB ? (size_t)(NT / 16 + 7) * 1024 : 0);
    const int C = (N1 > 16) ? Big::C : 16;   // columns per A task
    const bool tc = kTcOk && s->tc_stage;
    const size_t smem_tc = smem > kTcSmem ? smem : kTcSmem;
    if (query) {
        int rc = prep_smem(kern, smem);
        if (rc) return rc;
        if (kTcOk) { rc = prep_smem(kern_tc, smem_tc); if (rc) return rc; }
        if constexpr (kF2) { rc = prep_smem(k_fused2<PL, MODE_PFB, N1>, Fused2Shape<PL, MODE_PFB, N1>::SMEM); if (rc) return rc; }
        // resident CTAs per SM: 128 registers x 512 threads fill the register file, 4 x 64 (2 x 128) TMEM
        // columns and 4 x 33 KB of shared memory fit.  The occupancy API cannot be asked: it reports 1
        // for any kernel that contains tcgen05.alloc (measured: 4 such CTAs of 128 threads do share an
        // SM), which also rules out cudaLaunchCooperativeKernel for a grid of this size.
        const int per_sm = PER_SM;
        s->fgrid = per_sm * s->numSM;
        return 0;
    }
    auto ilog2 = [](int v) { int l = 0; while ((1 << l) < v) l++; return l; };
    const int ngroups = (int)((nspec + s->fGS - 1) / s->fGS);
    if (ngroups > s->fcap) {   // a longer call than spec_create sized the counters for (rare)
        if (s->capturing) return SPEC_ERR_STATE;
        CK(cudaStreamSynchronize(st));
        int rc = fused_alloc_flags(s, ngroups);
        if (rc) return rc;
    }
    // consecutive launches may overlap (programmatic dependent launch): they alternate between two Z rings
    // and two sets of counters
    const int par = s->fpar;
    unsigned* const flags = s->d_flags + (size_t)par * (FUSED_ROLE_WORDS + 2 * s->fcap);
    FusedParams p;
    p.view = view; p.h = s->d_coef; p.Z = s->d_Z + (size_t)(s->fpdl ? par : 0) * s->zbatch * s->N;
    p.twN = s->d_twN; p.twT = s->d_twT; p.tw1 = s->d_tw1; p.twL = s->d_tw2;
    p.ring = s->d_ring; p.acc_stride = acc_floats(s); p.nring = s->nring;
    p.N = s->N; p.N2 = s->N2; p.nspec = (int)nspec; p.c0 = c0; p.M = s->M;
    p.lgGS = ilog2(s->fGS); p.RING = s->fRING; p.lgTPG = ilog2(s->N2 / C); p.na_per_sm = s->fna; p.per_sm = PER_SM;
    p.role = flags; p.a_done = flags + FUSED_ROLE_WORDS; p.b_done = flags + FUSED_ROLE_WORDS + s->fcap;
    p.err = s->d_err;
    p.carry_src = (const uint4*)s->carry_src; p.carry_dst = (uint4*)s->carry_dst; p.carry_chunks = (int)(s->carry_bytes / 16);
    p.carry_cnt = s->d_carry_cnt; p.carry_wait = s->carry_cum; p.carry_wait_on = (s->hist_by_kernel && view.nhist > 0) ? 1 : 0;
    // Captured into a CUDA graph: the launches of the segment do not overlap (plain dependencies order the history
    // hand-over) and the carry counter's absolute target would be stale at replay, so neither is used.
    if (s->capturing) p.carry_wait_on = 0;
    p.dump = s->dump;
    p.tcB = s->d_tcB;
#ifdef SPEC_TUNING
    p.na_per_sm = tuning_int("SPEC_FUSED_NA", p.na_per_sm, 1, PER_SM - 1);
#endif
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(s->fgrid); cfg.blockDim = dim3(NT); cfg.dynamicSmemBytes = tc ? smem_tc : smem; cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at; cfg.numAttrs = (s->fpdl && !s->capturing) ? 1 : 0;
    if (s->dump) {   // test hook: the same kernel, front end only (no carry, no accumulation)
        auto kd = k_fused<PL, NT, MODE_PFB, PER_SM, true, N1>;
        int rc = prep_smem(kd, smem);
        if (rc) return rc;
        p.carry_chunks = 0; p.carry_wait_on = 0;
        cfg.numAttrs = 0;
        cfg.dynamicSmemBytes = smem;
        CK(cudaLaunchKernelEx(&cfg, kd, p));
        CK(cudaGetLastError());
        return 0;
    }
    {
        FusedChain& ch = fused_chain();
        std::lock_guard<std::mutex> lk(ch.mu);
        int rc = fused_chain_enter(ch, st);
        if (rc) return rc;
        {
            ProfScope ps(s, 0, st);
            if (tc) CK(cudaLaunchKernelEx(&cfg, kern_tc, p));
            else if constexpr (kF2) {
                typedef Fused2Shape<PL, MODE_PFB, N1> SH2;
                cfg.gridDim = dim3((256 / SH2::NT) * s->numSM); cfg.blockDim = dim3(2 * SH2::NT);
                cfg.dynamicSmemBytes = SH2::SMEM;
                CK(cudaLaunchKernelEx(&cfg, k_fused2<PL, MODE_PFB, N1>, p));
            } else CK(cudaLaunchKernelEx(&cfg, kern, p));
        }
        CK(cudaGetLastError());
        rc = fused_chain_leave(ch, st);
        if (rc) return rc;
    }
    // the launch is queued: only now does the handle move on
    s->fpar ^= 1;
    if (p.carry_chunks) s->carry_cum += cfg.gridDim.x;
    return 0;
}

static int fused_dispatch(spec_ctx* s, bool query, const InputView& view, long long nspec, long long c0, cudaStream_t st) {
    const bool pfb = (s->mode == SPEC_MODE_PFB);
    switch (s->N1) {   // N >= 131072: N1 x 4096
#define FB_CASE(N1V)                                                                      \
    case N1V:                                                                             \
        return pfb ? fused_do<PL4096, 256, 1, 2, N1V>(s, query, view, nspec, c0, st)      \
                   : fused_do<PL4096, 256, 0, 2, N1V>(s, query, view, nspec, c0, st);
        FB_CASE(32)
        FB_CASE(64)
        FB_CASE(128)
#undef FB_CASE
    }
    switch (s->N2) {
#define F_CASE(LEN, PLX, NT, PS)                                                     \
    case LEN:                                                                        \
        return pfb ? fused_do<PLX, NT, 1, PS>(s, query, view, nspec, c0, st)         \
                   : fused_do<PLX, NT, 0, PS>(s, query, view, nspec, c0, st);
        F_CASE(512, PL512, 128, FUSED_PER_SM)
        F_CASE(1024, PL1024, 128, FUSED_PER_SM)
        F_CASE(2048, PL2048, 128, FUSED_PER_SM)
        F_CASE(4096, PL4096, 256, 2)
#undef F_CASE
        case 64: return fused_do<PL64, 128, 1, FUSED_PER_SM>(s, query, view, nspec, c0, st);
        case 128: return fused_do<PL128, 128, 1, FUSED_PER_SM>(s, query, view, nspec, c0, st);
        case 256: return fused_do<PL256, 128, 1, FUSED_PER_SM>(s, query, view, nspec, c0, st);
    }
    return SPEC_ERR_ARG;
}

// `nspec` spectra starting at view-spectrum m0; c0 = spectra produced before them (window bookkeeping
// is done inside the kernels, so a launch may span accumulation windows)
// Packet-sized calls: a persistent launch costs about 8-11 us however little it has to do
// (every CTA of a whole-GPU grid allocates tensor memory, waits for all the others, carries history, drains); below this many
// samples the same 16 x N2 plan runs as two ordinary launches instead (pass A into the Z ring's memory, pass B out of it):
// same intermediate layout, same accumulator order, so calls of both kinds mix freely on one handle.
static bool small_call(const spec_ctx* s, long long nspec) {
    return s->fused && s->N1 == 16 && !s->dump && !s->tc_stage && nspec * (long long)s->N <= (1ll << 18) && nspec <= s->zbatch;
}

static int run_spectra(spec_ctx* s, const InputView& v, long long m0, long long nspec, long long c0, cudaStream_t st) {
    if (s->N1 == 1) return run_single(s, v, m0, nspec, c0, st);
    if (small_call(s, nspec) && (s->mode == SPEC_MODE_PFB || !s->use_coef)) {
        int rc = run_passA(s, v, m0, (int)nspec, st);
        if (rc) return rc;
        return run_passB(s, (int)nspec, c0, st);
    }
    if (s->r2_single) return s->use_coef ? launch_single_r2<PL4096, 1>(s, v, nspec, c0, st) : launch_single_r2<PL4096, 0>(s, v, nspec, c0, st);
    if (s->fused && (s->mode == SPEC_MODE_PFB || !s->use_coef)) return fused_dispatch(s, false, v, nspec, c0, st);
    for (long long b0 = 0; b0 < nspec; b0 += s->zbatch) {
        const int nb = (int)((nspec - b0 < s->zbatch) ? nspec - b0 : s->zbatch);
        int rc = run_passA(s, v, m0 + b0, nb, st);
        if (rc) return rc;
        rc = run_passB(s, nb, c0 + b0, st);
        if (rc) return rc;
    }
    return 0;
}

// ------------------------------------------------------------------ API
static void free_all(spec_ctx* s) {
    prof_fold(s);
    for (auto e : s->pool) cudaEventDestroy(e);
    cudaFree(s->d_coef); cudaFree(s->d_twN); cudaFree(s->d_twT); cudaFree(s->d_tcB); cudaFree(s->d_tw1); cudaFree(s->d_tw2); cudaFree(s->d_perm);
    cudaFree(s->d_hist[0]); cudaFree(s->d_hist[1]); cudaFree(s->d_hist[2]); cudaFree(s->d_carry_cnt); cudaFree(s->d_Z); cudaFree(s->d_Y); cudaFree(s->d_ring); cudaFree(s->d_stage);
    cudaFree(s->d_sbuf[0]); cudaFree(s->d_sbuf[1]); cudaFree(s->d_flags);
    if (s->h_err) cudaFreeHost(s->h_err);
    if (s->side) cudaStreamDestroy(s->side);
    for (int i = 0; i < 2; i++) {
        if (s->ev_copied[i]) cudaEventDestroy(s->ev_copied[i]);
        if (s->ev_used[i]) cudaEventDestroy(s->ev_used[i]);
    }
}

static int alloc_ring(spec_ctx* s, int nslots) {
    float* r = nullptr;
    CK(cudaMalloc(&r, (size_t)(nslots + 1) * acc_floats(s) * sizeof(float)));
    CK(cudaMemset(r, 0, (size_t)(nslots + 1) * acc_floats(s) * sizeof(float)));   // slots stay zero while free (k_unpermute clears)
    cudaFree(s->d_ring);
    s->d_ring = r;
    s->nring = nslots + 1;
    return 0;
}

static int create_impl(spec_ctx* s) {
    int dev = 0;
    CK(cudaGetDevice(&dev));
    CK(cudaDeviceGetAttribute(&s->numSM, cudaDevAttrMultiProcessorCount, dev));
    const int N = s->N;
    // four-step split: one kernel up to 4096 channels, N1 x N2 beyond
    // fused persistent kernel (fused.cuh): dual-pol, 16 x N2, PFB with the paper's 8 taps from 1024
    // channels (the FIR needs the column split to reuse each unpacked sample), direct FFT from 8192
    int regs_per_sm = 0, cc_major = 0;
    CK(cudaDeviceGetAttribute(&regs_per_sm, cudaDevAttrMaxRegistersPerMultiprocessor, dev));
    CK(cudaDeviceGetAttribute(&cc_major, cudaDevAttrComputeCapabilityMajor, dev));
    // (the resident-grid arithmetic of the fused kernel assumes the 64 K-register SM of sm_100)
    s->fused = regs_per_sm == 65536 && cc_major == 10 &&
               s->P == 2 && N >= 1024 &&
               ((s->mode == SPEC_MODE_PFB && s->T == 8) || (s->mode == SPEC_MODE_FFT && N >= 8192));
#ifdef SPEC_TUNING
    if (tuning_int("SPEC_NO_FUSED", 0, 0, 1)) s->fused = false;
#endif
    s->r2_single = cc_major == 10 && s->P == 2 && s->mode == SPEC_MODE_FFT && N == 8192;
    if (s->r2_single) { s->fused = false; s->N1 = 2; s->N2 = N / 2; }
    else if (s->fused && N <= 65536) { s->N1 = 16; s->N2 = N / 16; }
    else if (s->fused) { s->N2 = 4096; s->N1 = N / 4096; }
    else if (N <= 4096) { s->N1 = 1; s->N2 = N; }
    else if (N <= 65536) { s->N1 = 16; s->N2 = N / 16; }
    else { s->N2 = 4096; s->N1 = N / 4096; }

    default_coeffs(s, s->h_coef);
    CK(cudaMalloc(&s->d_coef, s->h_coef.size() * sizeof(float)));
    CK(cudaMemcpy(s->d_coef, s->h_coef.data(), s->h_coef.size() * sizeof(float), cudaMemcpyHostToDevice));
    s->use_coef = (s->mode == SPEC_MODE_PFB) || (s->window != SPEC_WINDOW_RECT);

    std::vector<float2> w;
    make_stage_twiddles(s->N2, w);
    CK(cudaMalloc(&s->d_tw2, w.size() * sizeof(float2)));
    CK(cudaMemcpy(s->d_tw2, w.data(), w.size() * sizeof(float2), cudaMemcpyHostToDevice));
    if (s->N1 > 1) {
        make_stage_twiddles(s->N1, w);
        CK(cudaMalloc(&s->d_tw1, w.size() * sizeof(float2)));
        CK(cudaMemcpy(s->d_tw1, w.data(), w.size() * sizeof(float2), cudaMemcpyHostToDevice));
        make_twiddles(N, w);
        CK(cudaMalloc(&s->d_twN, w.size() * sizeof(float2)));
        CK(cudaMemcpy(s->d_twN, w.data(), w.size() * sizeof(float2), cudaMemcpyHostToDevice));
        // two-launch path: the Z batch of one launch pair.  Measured (profiles/r01b_tuning.md): long runs per CTA
        // and few launches matter more here than keeping Z in L2, so the batch covers a whole 64 MiB call
        // (256 MiB of Z)
        size_t zmb = 256;
#ifdef SPEC_TUNING
        zmb = (size_t)tuning_int("SPEC_ZBATCH_MB", 256, 1, 4096);
#endif
        size_t zb = (zmb << 20) / ((size_t)N * sizeof(float4));
        s->zbatch = (int)(zb < 1 ? 1 : zb);
        if (s->fused) {
            InputView none{nullptr, nullptr, 0};
            int rc = fused_dispatch(s, true, none, 0, 0, nullptr);
            if (rc) return rc;
            const int NT = (s->N2 == 4096) ? 256 : 128;
            s->fGS = (s->N2 >= 512) ? 16 : 32;   // spectra per ring group (measured best in round 1)
            if (s->N1 > 16) s->fGS = (s->N1 == 128) ? 4 : 8;   // one producer phase per group (ProducerBig::R)
#ifdef SPEC_TUNING
            { const int v = tuning_int("SPEC_FUSED_GS", s->fGS, 2, 4096); if (!(v & (v - 1))) s->fGS = v; }
#endif
            // producer share of the resident CTAs: two of the four CTAs of an SM produce, in both modes.  The
            // FIR makes an A task about as long as the row FFT of the same samples; without it (direct-FFT
            // mode) one producer per SM was the first choice, but two measure faster now that consecutive
            // launches overlap (round 1: N=8192 101 -> 115 GHz, N=32768 111 -> 112 GHz)
            s->fna = (NT == 256) ? 1 : 2;
            // ring = what the producers (one task each) and the consumers (one job of 16*NT points each)
            // hold at a time, plus two groups of slack
            const int per_sm = (NT == 256) ? 2 : FUSED_PER_SM, nsm = s->fgrid / per_sm;
            const int tpg = s->N2 / 16;
            const int a_groups = (nsm * s->fna + tpg - 1) / tpg;
            const long long b_spectra = ((long long)nsm * (per_sm - s->fna) * NT * 16 + N - 1) / N;
            s->fRING = a_groups + (int)((b_spectra + s->fGS - 1) / s->fGS) + 2;
            if (s->N1 > 16) {
                // N >= 131072: the consumers all work on one spectrum at a time (one row each), the producers on
                // one group; the ring holds the group being read, the one being written and one of slack while that
                // still fits the L2 (a 2^19-point dual-pol spectrum is 8 MiB of Z).  One ring only: consecutive
                // launches do not overlap here.
                const size_t group_bytes = (size_t)s->fGS * N * sizeof(float4);
                s->fRING = (3 * group_bytes <= ((size_t)48 << 20)) ? 3 : 2;
                s->fpdl = 0;
            }
#ifdef SPEC_TUNING
            s->fRING = tuning_int("SPEC_FUSED_RING", s->fRING, 2, 4096);
            s->fpdl = tuning_int("SPEC_FUSED_PDL", s->fpdl, 0, 1);
#endif
            s->zbatch = s->fRING * s->fGS;
            CK(cudaHostAlloc(&s->h_err, sizeof(unsigned), cudaHostAllocMapped));
            *s->h_err = 0u;
            CK(cudaHostGetDevicePointer(&s->d_err, s->h_err, 0));
            CK(cudaMalloc(&s->d_carry_cnt, sizeof(unsigned)));
            CK(cudaMemset(s->d_carry_cnt, 0, sizeof(unsigned)));
            // per-group counters for calls of up to 2^28 samples (1 GiB of dual-pol input); a longer call grows them
            rc = fused_alloc_flags(s, (int)(((1ll << 28) / N + s->fGS - 1) / s->fGS));
            if (rc) return rc;
        }
        // (fused path: two rings, alternating launches may overlap)
        if (!s->r2_single) CK(cudaMalloc(&s->d_Z, (size_t)((s->fused && s->fpdl) ? 2 : 1) * s->zbatch * N * sizeof(float4)));
        if (s->fused && s->N1 > 16) {
            std::vector<float2> wt((size_t)N);
            for (int p1 = 0; p1 < s->N1; p1++) {
                const long k1 = pos_to_freq(s->N1, p1);
                for (int n2 = 0; n2 < s->N2; n2++) {
                    const double a = -2.0 * M_PI * (double)((k1 * n2) % N) / (double)N;
                    wt[(size_t)p1 * s->N2 + n2] = make_float2((float)cos(a), (float)sin(a));
                }
            }
            CK(cudaMalloc(&s->d_twT, wt.size() * sizeof(float2)));
            CK(cudaMemcpy(s->d_twT, wt.data(), wt.size() * sizeof(float2), cudaMemcpyHostToDevice));
        }
        if (s->fused) {
            // Residency probe: the persistent grid assumes PER_SM CTAs on every SM at once (nothing can ask the
            // occupancy API, see fused_do).  An empty launch of the same kernel proves it here: every CTA waits for
            // all the others to arrive; if they cannot (an SM limit, a long-running foreign kernel) the wait
            // expires, the error word is raised and this handle falls back to the two-launch path.
            InputView none{nullptr, nullptr, 0};
            int prc = fused_dispatch(s, false, none, 0, 0, nullptr);
            if (prc == 0) {
                CK(cudaDeviceSynchronize());
                if (*(volatile unsigned*)s->h_err) prc = SPEC_ERR_CUDA;
            }
            if (prc) {
                *s->h_err = 0u;
                CK(cudaMemset(s->d_flags, 0, (size_t)2 * (FUSED_ROLE_WORDS + 2 * s->fcap) * sizeof(unsigned)));
                s->fused = false;
                s->fpar = 0;
                cudaFree(s->d_Z);
                s->d_Z = nullptr;
                size_t zb2 = ((size_t)256 << 20) / ((size_t)N * sizeof(float4));
                s->zbatch = (int)(zb2 < 1 ? 1 : zb2);
                CK(cudaMalloc(&s->d_Z, (size_t)s->zbatch * N * sizeof(float4)));
            }
        }
        if (!s->fused && s->mode == SPEC_MODE_PFB && s->T == 8 && s->N1 > 16)
            CK(cudaMalloc(&s->d_Y, (size_t)s->zbatch * N * sizeof(float4)));
    }
    std::vector<int> perm(N);
    for (int a = 0; a < N; a++) {
        const int p1 = a / s->N2, p2 = a % s->N2;
        perm[a] = pos_to_freq(s->N1, p1) + s->N1 * pos_to_freq(s->N2, p2);
    }
    CK(cudaMalloc(&s->d_perm, (size_t)N * sizeof(int)));
    CK(cudaMemcpy(s->d_perm, perm.data(), (size_t)N * sizeof(int), cudaMemcpyHostToDevice));

    if (s->T > 1)
        for (int i = 0; i < 3; i++) CK(cudaMalloc(&s->d_hist[i], (size_t)(s->T - 1) * block_bytes(s)));
    int rc = alloc_ring(s, 8);
    if (rc) return rc;
    CK(cudaMalloc(&s->d_stage, acc_floats(s) * sizeof(float)));
    return 0;
}

extern "C" int spec_create(spec_t** out, int nchan, int ntaps, int npol, int mode, long nacc, int window) {
    if (!out) return SPEC_ERR_ARG;
    if (nchan < 16 || nchan > 524288 || (nchan & (nchan - 1))) return SPEC_ERR_ARG;
    if (npol != 1 && npol != 2) return SPEC_ERR_ARG;
    if (mode != SPEC_MODE_PFB && mode != SPEC_MODE_FFT) return SPEC_ERR_ARG;
    if (window != SPEC_WINDOW_RECT && window != SPEC_WINDOW_HANN) return SPEC_ERR_ARG;
    if (nacc < 1) return SPEC_ERR_ARG;
    if (mode == SPEC_MODE_FFT) ntaps = 1;
    if (ntaps < 1 || ntaps > 64) return SPEC_ERR_ARG;
    spec_ctx* s = new (std::nothrow) spec_ctx();
    if (!s) return SPEC_ERR_NOMEM;
    s->N = nchan; s->T = ntaps; s->P = npol; s->S = (npol == 2) ? 4 : 1;
    s->mode = mode; s->window = window; s->M = nacc;
    int rc = create_impl(s);
    if (rc) { free_all(s); delete s; return rc; }
    *out = s;
    return SPEC_OK;
}

extern "C" int spec_destroy(spec_t* s);

extern "C" int spec_create_subbands(spec_t** out, int nsub, int nchan, int ntaps, int npol, int mode, long nacc, int window) {
    if (!out || nsub < 1 || nsub > 16) return SPEC_ERR_ARG;
    if (nsub == 1) return spec_create(out, nchan, ntaps, npol, mode, nacc, window);
    spec_ctx* p = new (std::nothrow) spec_ctx();
    if (!p) return SPEC_ERR_NOMEM;
    p->nsub = nsub;
    for (int i = 0; i < nsub; i++) {
        spec_ctx* c = nullptr;
        int rc = spec_create(&c, nchan, ntaps, npol, mode, nacc, window);
        if (rc) { spec_destroy(p); return rc; }
        p->subs.push_back(c);
    }
    // what the parent's own entry points look at
    p->N = nchan; p->P = npol; p->S = p->subs[0]->S; p->T = p->subs[0]->T; p->mode = mode; p->window = window; p->M = nacc;
    *out = p;
    return SPEC_OK;
}

extern "C" int spec_destroy(spec_t* s) {
    if (!s) return SPEC_ERR_ARG;
    if (s->nsub > 1) {
        for (auto c : s->subs) spec_destroy(c);
        cudaFree(s->d_deint);
        cudaFree(s->d_sbuf[0]); cudaFree(s->d_sbuf[1]);
        if (s->side) cudaStreamDestroy(s->side);
        for (int i = 0; i < 2; i++) {
            if (s->ev_copied[i]) cudaEventDestroy(s->ev_copied[i]);
            if (s->ev_used[i]) cudaEventDestroy(s->ev_used[i]);
        }
        delete s;
        return SPEC_OK;
    }
    cudaDeviceSynchronize();
    if (s->fused) fused_chain_quiesce();
    free_all(s);
    delete s;
    return SPEC_OK;
}

extern "C" int spec_set_coeffs(spec_t* s, const float* h, size_t count) {
    if (!s || !h) return SPEC_ERR_ARG;
    if (s->nsub > 1) {   // every sub-band runs the same filter
        for (auto c : s->subs) { int rc = spec_set_coeffs(c, h, count); if (rc) return rc; }
        return SPEC_OK;
    }
    if (count != s->h_coef.size()) return SPEC_ERR_SIZE;
    CK(cudaDeviceSynchronize());
    CK(cudaMemcpy(s->d_coef, h, count * sizeof(float), cudaMemcpyHostToDevice));
    s->h_coef.assign(h, h + count);
    s->use_coef = true;
    if (s->mode == SPEC_MODE_FFT) {   // an all-ones window is the rectangular one: no multiply, same plan as RECT
        bool ones = true;
        for (size_t i = 0; i < count && ones; i++) ones = (h[i] == 1.0f);
        if (ones) s->use_coef = false;
    }
    return SPEC_OK;
}

extern "C" int spec_get_coeffs(const spec_t* s, float* h_out, size_t count) {
    if (!s || !h_out) return SPEC_ERR_ARG;
    if (s->nsub > 1) return spec_get_coeffs(s->subs[0], h_out, count);
    if (count != s->h_coef.size()) return SPEC_ERR_SIZE;
    memcpy(h_out, s->h_coef.data(), count * sizeof(float));
    return SPEC_OK;
}

// The split fp16 DFT matrix B' of fused_producer_fft_tc: [split][k/8][col/8][col%8][k%8], k = pol*32 + 2 n1 + c,
// col = 4 k1 + {Xre, Yre, Xim, Yim}; X[k1] = sum_n1 x[n1] exp(-2 pi i n1 k1 / 16)
static void make_tc_matrix(std::vector<__half>& out) {
    out.assign((size_t)kTcSplit * 64 * 64, __float2half_rn(0.f));
    for (int col = 0; col < 64; col++)
        for (int kk = 0; kk < 64; kk++) {
            const int k1 = col >> 2, j = col & 3, pol = j & 1, c_out = j >> 1;
            const int pol_in = kk >> 5, n1 = (kk & 31) >> 1, c_in = kk & 1;
            double v = 0.0;
            if (pol_in == pol) {
                const double th = 2.0 * M_PI * (double)((n1 * k1) % 16) / 16.0;
                const double cs = cos(th), sn = sin(th);
                v = (c_out == 0) ? (c_in == 0 ? cs : sn) : (c_in == 0 ? -sn : cs);
            }
            if (fabs(v) < 1e-12) v = 0.0;
            double rem = v;
            for (int sp = 0; sp < kTcSplit; sp++) {
                const __half h = __float2half_rn((float)rem);
                rem -= (double)__half2float(h);
                out[(size_t)sp * 4096 + (size_t)(kk >> 3) * 512 + (size_t)(col >> 3) * 64 + (size_t)(col & 7) * 8 + (kk & 7)] = h;
            }
        }
}

static int fused_failed(spec_ctx* s);

// ---- CUDA-graph capture of a periodic call sequence
extern "C" int spec_capture_begin(spec_t* s) {
    if (!s) return SPEC_ERR_ARG;
    if (s->nsub > 1) return SPEC_ERR_STATE;   // per-sub-band handles only
    if (fused_failed(s)) return SPEC_ERR_CUDA;
    if (s->capturing || s->prof) return SPEC_ERR_STATE;
    if (windows_done(s) != s->win_read) return SPEC_ERR_STATE;   // read what is pending first
    s->capturing = true;
    s->cap_cur = s->cur; s->cap_fpar = s->fpar; s->cap_nhist = s->nhist;
    s->cap_count = s->count; s->cap_win_read = s->win_read;
    return SPEC_OK;
}

extern "C" int spec_capture_end(spec_t* s) {
    if (!s) return SPEC_ERR_ARG;
    if (s->nsub > 1) return SPEC_ERR_STATE;   // per-sub-band handles only
    if (!s->capturing) return SPEC_ERR_STATE;
    s->capturing = false;
    const long long dcount = s->count - s->cap_count, dwin = s->win_read - s->cap_win_read;
    // replayable only if every kernel argument baked into the graph is valid again at the end of the segment
    const bool periodic = s->cur == s->cap_cur && s->fpar == s->cap_fpar && s->nhist == s->cap_nhist &&
                          dcount % (s->M * (long long)s->nring) == 0 && windows_done(s) == s->win_read;
    if (!periodic) { s->cap_dcount = 0; s->cap_dwin = 0; return SPEC_ERR_STATE; }
    s->cap_dcount = dcount; s->cap_dwin = dwin;
    return SPEC_OK;
}

extern "C" int spec_replayed(spec_t* s, long times) {
    if (!s || times < 0) return SPEC_ERR_ARG;
    if (s->nsub > 1) return SPEC_ERR_STATE;   // per-sub-band handles only
    if (s->capturing || s->cap_dcount == 0) return SPEC_ERR_STATE;
    s->count += s->cap_dcount * times;
    s->win_read += s->cap_dwin * times;
    return SPEC_OK;
}

extern "C" int spec_accumulate_host(double* h_acc, const float* h_spectrum, size_t count) {
    if (!h_acc || !h_spectrum) return SPEC_ERR_ARG;
    for (size_t i = 0; i < count; i++) h_acc[i] += (double)h_spectrum[i];
    return SPEC_OK;
}

extern "C" int spec_set_option(spec_t* s, int option, int value) {
    if (!s) return SPEC_ERR_ARG;
    if (s->nsub > 1) {
        for (auto c : s->subs) { int rc = spec_set_option(c, option, value); if (rc) return rc; }
        return SPEC_OK;
    }
    if (option == SPEC_OPT_TENSOR_CORE_STAGE) {
        if (value != 0 && value != 1) return SPEC_ERR_ARG;
        // direct-FFT mode, rectangular window, dual-pol, 8192 <= nchan <= 32768 (the 16 x N2 plans of 128 threads)
        const bool ok = s->fused && s->mode == SPEC_MODE_FFT && s->N1 == 16 && s->N2 <= 2048;
        if (!ok) return value ? SPEC_ERR_STATE : SPEC_OK;
        if (value && !s->d_tcB) {
            std::vector<__half> b;
            make_tc_matrix(b);
            CK(cudaMalloc(&s->d_tcB, b.size() * sizeof(__half)));
            CK(cudaMemcpy(s->d_tcB, b.data(), b.size() * sizeof(__half), cudaMemcpyHostToDevice));
        }
        s->tc_stage = value != 0;
        return SPEC_OK;
    }
    return SPEC_ERR_ARG;
}

extern "C" int spec_pending(const spec_t* s) {
    if (!s) return SPEC_ERR_ARG;
    if (s->nsub > 1) return spec_pending(s->subs[0]);
    return (int)(windows_done(s) - s->win_read);
}
extern "C" long spec_spectra_done(const spec_t* s) {
    if (!s) return SPEC_ERR_ARG;
    if (s->nsub > 1) return spec_spectra_done(s->subs[0]);
    return (long)s->count;
}

extern "C" int spec_reset(spec_t* s) {
    if (!s) return SPEC_ERR_ARG;
    if (s->nsub > 1) {
        for (auto c : s->subs) { int rc = spec_reset(c); if (rc) return rc; }
        return SPEC_OK;
    }
    CK(cudaDeviceSynchronize());
    if (s->fused) fused_chain_quiesce();
    s->nhist = 0; s->cur = 0; s->count = 0; s->win_read = 0;
    s->carry_bytes = 0; s->hist_by_kernel = false; s->fpar = 0;
    if (s->failed || (s->h_err && *s->h_err)) {   // a failed or timed-out launch leaves its counters dirty
        if (s->h_err) *s->h_err = 0u;
        if (s->d_flags) CK(cudaMemset(s->d_flags, 0, (size_t)2 * (FUSED_ROLE_WORDS + 2 * s->fcap) * sizeof(unsigned)));
    }
    if (s->d_carry_cnt) CK(cudaMemset(s->d_carry_cnt, 0, sizeof(unsigned)));
    s->carry_cum = 0;
    CK(cudaMemset(s->d_ring, 0, (size_t)s->nring * acc_floats(s) * sizeof(float)));
    s->failed = false;
    return SPEC_OK;
}

extern "C" int spec_set_ring(spec_t* s, int nslots) {
    if (!s || nslots < 1 || nslots > 65536) return SPEC_ERR_ARG;
    if (s->nsub > 1) {
        for (auto c : s->subs) { int rc = spec_set_ring(c, nslots); if (rc) return rc; }
        return SPEC_OK;
    }
    if (s->count != 0 || s->nhist != 0) return SPEC_ERR_STATE;
    CK(cudaDeviceSynchronize());
    return alloc_ring(s, nslots);
}

static int fused_failed(spec_ctx* s) {
    if (s->h_err && *(volatile unsigned*)s->h_err) {
        snprintf(g_err, sizeof(g_err), "a wait inside the persistent kernel timed out (grid not fully resident?); "
                                       "results since the last spec_reset are invalid");
        return 1;
    }
    if (s->failed) {
        snprintf(g_err, sizeof(g_err), "an earlier spec_process failed part-way (CUDA error); call spec_reset");
        return 1;
    }
    return 0;
}

// eight-sub-band modes: split the interleaved input into one contiguous stream per sub-band, then run every
// sub-band's own chain on it (16 transforms per spectrum set, PAPER.md:90 step 1b) on the same stream
static int subbands_process(spec_ctx* p, const void* d_in, size_t nsamples, cudaStream_t st) {
    if (nsamples % (size_t)p->N) return SPEC_ERR_SIZE;
    if (nsamples == 0) return 0;
    if (!d_in || ((uintptr_t)d_in & 15)) return SPEC_ERR_ARG;
    for (auto c : p->subs) {   // nothing is queued unless every sub-band accepts the call
        if (fused_failed(c)) return SPEC_ERR_CUDA;
        const long long total = c->nhist + (long long)(nsamples / (size_t)c->N);
        const long long nspec = total >= c->T ? total - (c->T - 1) : 0;
        if ((c->count + nspec) / c->M - c->win_read > c->nring - 1) return SPEC_ERR_OVERRUN;
    }
    const size_t wbytes = (size_t)2 * p->P;
    if (nsamples > p->deint_cap) {
        cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
        if (cudaStreamIsCapturing(st, &cap) == cudaSuccess && cap != cudaStreamCaptureStatusNone) return SPEC_ERR_STATE;
        CK(cudaDeviceSynchronize());
        uint8_t* nb = nullptr;
        CK(cudaMalloc(&nb, nsamples * wbytes * p->nsub));
        cudaFree(p->d_deint);
        p->d_deint = nb;
        p->deint_cap = nsamples;
    }
    const int gx = cdiv((long long)nsamples, 256);
    if (p->P == 2)
        k_deinterleave<uint32_t><<<gx, 256, 0, st>>>((const uint32_t*)d_in, (uint32_t*)p->d_deint, nsamples, p->nsub, p->deint_cap);
    else
        k_deinterleave<uint16_t><<<gx, 256, 0, st>>>((const uint16_t*)d_in, (uint16_t*)p->d_deint, nsamples, p->nsub, p->deint_cap);
    CK(cudaGetLastError());
    int completed = 0;
    for (int i = 0; i < p->nsub; i++) {
        const int rc = spec_process(p->subs[i], p->d_deint + (size_t)i * p->deint_cap * wbytes, nsamples, st);
        if (rc < 0) return rc;
        completed = rc;
    }
    return completed;
}

extern "C" int spec_process(spec_t* s, const void* d_in, size_t nsamples, void* cuda_stream) {
    if (!s) return SPEC_ERR_ARG;
    if (s->nsub > 1) return subbands_process(s, d_in, nsamples, (cudaStream_t)cuda_stream);
    if (fused_failed(s)) return SPEC_ERR_CUDA;
    if (nsamples % (size_t)s->N) return SPEC_ERR_SIZE;
    if (nsamples == 0) return 0;
    if (!d_in || ((uintptr_t)d_in & 15)) return SPEC_ERR_ARG;  // bulk copies need 16-byte alignment
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const int T = s->T;
    const long long nblk = (long long)(nsamples / (size_t)s->N);
    const long long total = s->nhist + nblk;
    const long long nspec = total >= T ? total - (T - 1) : 0;
    const long long done_after = (s->count + nspec) / s->M;
    if (done_after - s->win_read > s->nring - 1) return SPEC_ERR_OVERRUN;
    const int completed = (int)(done_after - windows_done(s));
    // Everything above leaves the handle untouched.  From here on work is queued: a CUDA failure below marks the
    // handle failed (partly updated accumulators cannot be rolled back) until spec_reset.

    InputView view{s->d_hist[s->cur], (const uint8_t*)d_in, s->nhist};
    const int nxt = (s->cur + 1) % 3;
    const long long c = s->count + nspec;
    // carry the last min(T-1,total) blocks of  history ++ input  (reading R4).  On the fused path
    // the launch copies them itself when they all come from this call's input, so that consecutive launches
    // stay adjacent in the stream (programmatic dependent launch, fused.cuh).
    const long long keep = total < T - 1 ? total : T - 1;
    bool carried = false;
    if (nspec > 0) {
        if (s->fused && s->N1 > 1 && keep > 0 && nblk >= keep && (s->mode == SPEC_MODE_PFB || !s->use_coef) && !small_call(s, nspec)) {
            const size_t bb = block_bytes(s);
            s->carry_src = (const uint8_t*)d_in + (size_t)(nblk - keep) * bb;
            s->carry_dst = s->d_hist[nxt];
            s->carry_bytes = (size_t)keep * bb;
            carried = true;
        }
        int rc = run_spectra(s, view, 0, nspec, s->count, st);
        s->carry_bytes = 0;
        if (rc) { s->failed = true; return rc; }
    }
    if (carried) {
        s->cur = nxt;
        s->hist_by_kernel = true;
    } else if (keep > 0) {
        const size_t bb = block_bytes(s);
        uint8_t* dst = s->d_hist[nxt];
        const long long first = total - keep;
        long long nold = s->nhist - first;  // blocks still taken from the old history
        if (nold < 0) nold = 0;
        cudaError_t e = cudaSuccess;
        if (nold > 0)
            e = cudaMemcpyAsync(dst, s->d_hist[s->cur] + (size_t)first * bb, (size_t)nold * bb, cudaMemcpyDeviceToDevice, st);
        const long long nnew = keep - nold;
        if (e == cudaSuccess && nnew > 0)
            e = cudaMemcpyAsync(dst + (size_t)nold * bb, (const uint8_t*)d_in + (size_t)(nblk - nnew) * bb,
                                (size_t)nnew * bb, cudaMemcpyDeviceToDevice, st);
        if (e != cudaSuccess) { s->failed = true; return fail_cuda(e, "cudaMemcpyAsync(history)"); }
        s->cur = nxt;
        s->hist_by_kernel = false;   // ordinary stream order covers these copies
    }
    s->nhist = (int)keep;
    s->count = c;
    return completed;
}

extern "C" int spec_read_accum(spec_t* s, float* dst, int dst_is_device, void* cuda_stream) {
    if (!s || !dst) return SPEC_ERR_ARG;
    if (s->nsub > 1) {   // [nsub][S][nchan]
        int got = 0;
        for (int i = 0; i < s->nsub; i++) {
            got = spec_read_accum(s->subs[i], dst + (size_t)i * s->S * s->N, dst_is_device, cuda_stream);
            if (got <= 0) return got;
        }
        return got;
    }
    if (fused_failed(s)) return SPEC_ERR_CUDA;
    if (windows_done(s) - s->win_read <= 0) return 0;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    float* out = dst_is_device ? dst : s->d_stage;
    {
        ProfScope ps(s, 3, st);
        k_unpermute<<<cdiv(s->N, 256), 256, 0, st>>>(s->d_ring, s->d_perm, out, s->N, s->S,
                                                     (int)(s->win_read % s->nring), s->nring);
    }
    CK(cudaGetLastError());
    if (!dst_is_device) {
        CK(cudaMemcpyAsync(dst, s->d_stage, acc_floats(s) * sizeof(float), cudaMemcpyDeviceToHost, st));
        CK(cudaStreamSynchronize(st));
    }
    s->win_read++;
    return 1;
}

extern "C" int spec_read_accum_batch(spec_t* s, float* d_dst, int max_count, void* cuda_stream) {
    if (!s || !d_dst || max_count < 0) return SPEC_ERR_ARG;
    if (s->nsub > 1) {   // [count][nsub][S][nchan]
        int n = spec_pending(s);
        if (n > max_count) n = max_count;
        for (int c = 0; c < n; c++)
            for (int i = 0; i < s->nsub; i++) {
                const int rc = spec_read_accum(s->subs[i], d_dst + ((size_t)c * s->nsub + i) * s->S * s->N, 1, cuda_stream);
                if (rc < 0) return rc;
            }
        return n;
    }
    if (fused_failed(s)) return SPEC_ERR_CUDA;
    long long n = windows_done(s) - s->win_read;
    if (n > max_count) n = max_count;
    if (n <= 0) return 0;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    {
        ProfScope ps(s, 3, st);
        k_unpermute<<<dim3(cdiv(s->N, 256), (unsigned)n), 256, 0, st>>>(s->d_ring, s->d_perm, d_dst, s->N, s->S,
                                                                        (int)(s->win_read % s->nring), s->nring);
    }
    CK(cudaGetLastError());
    s->win_read += n;
    return (int)n;
}

extern "C" int spec_stream_host(spec_t* s, const void* h_pinned, size_t nsamples, size_t chunk_samples,
                                void* cuda_stream) {
    if (!s || (!h_pinned && nsamples)) return SPEC_ERR_ARG;
    if (chunk_samples == 0 || chunk_samples % (size_t)s->N || nsamples % (size_t)s->N) return SPEC_ERR_SIZE;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const size_t bps = (size_t)2 * s->P * s->nsub;
    const size_t cbytes = chunk_samples * bps;
    if (!s->side) {
        CK(cudaStreamCreateWithFlags(&s->side, cudaStreamNonBlocking));
        for (int i = 0; i < 2; i++) {
            CK(cudaEventCreateWithFlags(&s->ev_copied[i], cudaEventDisableTiming));
            CK(cudaEventCreateWithFlags(&s->ev_used[i], cudaEventDisableTiming));
        }
    }
    if (s->sbuf_bytes < cbytes) {
        CK(cudaDeviceSynchronize());
        for (int i = 0; i < 2; i++) {
            cudaFree(s->d_sbuf[i]);
            s->d_sbuf[i] = nullptr;
            CK(cudaMalloc(&s->d_sbuf[i], cbytes));
        }
        s->sbuf_bytes = cbytes;
        for (int i = 0; i < 2; i++) CK(cudaEventRecord(s->ev_used[i], st));
    }
    int completed = 0;
    size_t done = 0;
    for (int i = 0; done < nsamples; i++) {
        const int b = i & 1;
        const size_t n = (nsamples - done < chunk_samples) ? nsamples - done : chunk_samples;
        // side stream: wait until the compute stream has finished with this buffer, then copy
        CK(cudaStreamWaitEvent(s->side, s->ev_used[b], 0));
        CK(cudaMemcpyAsync(s->d_sbuf[b], (const uint8_t*)h_pinned + done * bps, n * bps, cudaMemcpyHostToDevice,
                           s->side));
        CK(cudaEventRecord(s->ev_copied[b], s->side));
        CK(cudaStreamWaitEvent(st, s->ev_copied[b], 0));
        const int rc = spec_process(s, s->d_sbuf[b], n, st);
        if (rc < 0) return rc;
        completed += rc;
        CK(cudaEventRecord(s->ev_used[b], st));
        done += n;
    }
    return completed;
}

extern "C" int spec_measure_fp32_peak(double* out_tflops, void* cuda_stream) {
    if (!out_tflops) return SPEC_ERR_ARG;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int dev = 0, nsm = 0;
    CK(cudaGetDevice(&dev));
    CK(cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev));
    float* buf = nullptr;
    CK(cudaMalloc(&buf, (size_t)nsm * 1024 * sizeof(float)));
    cudaEvent_t e0, e1;
    CK(cudaEventCreate(&e0));
    CK(cudaEventCreate(&e1));
    const int iters = 16384;
    double best = 0.0;
    for (int rep = 0; rep < 4; rep++) {
        CK(cudaEventRecord(e0, st));
        k_fp32_peak<<<nsm, 1024, 0, st>>>(buf, iters, 0.999f, 0.001f);
        CK(cudaEventRecord(e1, st));
        CK(cudaEventSynchronize(e1));
        float ms = 0.f;
        CK(cudaEventElapsedTime(&ms, e0, e1));
        const double tf = 2.0 * 16.0 * iters * 1024.0 * nsm / (ms * 1e-3) / 1e12;
        if (rep > 0 && tf > best) best = tf;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(buf);
    *out_tflops = best;
    return SPEC_OK;
}

extern "C" int spec_debug_probe(int op, double* out_per_clk_sm, void* cuda_stream) {
    if (!out_per_clk_sm || op < 0 || op > 6) return SPEC_ERR_ARG;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int dev = 0, nsm = 0, khz = 0;
    CK(cudaGetDevice(&dev));
    CK(cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev));
    CK(cudaDeviceGetAttribute(&khz, cudaDevAttrClockRate, dev));
    float* buf = nullptr;
    CK(cudaMalloc(&buf, (size_t)nsm * 1024 * sizeof(float)));
    cudaEvent_t e0, e1;
    CK(cudaEventCreate(&e0));
    CK(cudaEventCreate(&e1));
    const int iters = 8192;
    static const double per_iter[7] = {16, 8, 8, 16, 4, 4, 16};
    auto launch = [&](void) {
        switch (op) {
            case 0: k_probe<0><<<nsm, 1024, 0, st>>>(buf, iters, 0.999f, 0.001f); break;
            case 1: k_probe<1><<<nsm, 1024, 0, st>>>(buf, iters, 0.999f, 0.001f); break;
            case 2: k_probe<2><<<nsm, 1024, 0, st>>>(buf, iters, 0.999f, 0.001f); break;
            case 3: k_probe<3><<<nsm, 1024, 0, st>>>(buf, iters, 0.999f, 0.001f); break;
            case 4: k_probe<4><<<nsm, 1024, 65536, st>>>(buf, iters, 0.999f, 0.001f); break;
            case 5: k_probe<5><<<nsm, 1024, 65536, st>>>(buf, iters, 0.999f, 0.001f); break;
            default: k_probe<6><<<nsm, 1024, 0, st>>>(buf, iters, 0.999f, 0.001f); break;
        }
    };
    CK(cudaFuncSetAttribute(k_probe<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, 65536));
    CK(cudaFuncSetAttribute(k_probe<5>, cudaFuncAttributeMaxDynamicSharedMemorySize, 65536));
    double best = 0.0;
    for (int rep = 0; rep < 3; rep++) {
        CK(cudaEventRecord(e0, st));
        launch();
        CK(cudaEventRecord(e1, st));
        CK(cudaEventSynchronize(e1));
        float ms = 0.f;
        CK(cudaEventElapsedTime(&ms, e0, e1));
        const double v = per_iter[op] * iters * 1024.0 / (ms * 1e-3) / ((double)khz * 1e3);
        if (rep > 0 && v > best) best = v;
    }
    CK(cudaGetLastError());
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(buf);
    *out_per_clk_sm = best;
    return SPEC_OK;
}

extern "C" int spec_debug_unpack(const void* d_bytes, size_t nbytes, int npol, float* d_out, void* cuda_stream) {
    if (!d_bytes || !d_out || (npol != 1 && npol != 2)) return SPEC_ERR_ARG;
    if (nbytes == 0) return SPEC_OK;
    k_debug_unpack<<<cdiv((long long)((nbytes + 3) / 4), 256), 256, 0, (cudaStream_t)cuda_stream>>>(
        (const uint8_t*)d_bytes, nbytes, d_out, npol);
    CK(cudaGetLastError());
    return SPEC_OK;
}

// Runs the FRONT END of the kernel this handle's plan uses (its own staging, index arithmetic, unpack and FIR /
// window code: a DUMP instantiation of the same kernel template) and writes what it hands to the first butterfly.
extern "C" int spec_debug_fir(spec_t* s, const void* d_blocks, int nspec, float* d_out, void* cuda_stream) {
    if (!s || !d_blocks || !d_out || nspec < 1 || ((uintptr_t)d_blocks & 15)) return SPEC_ERR_ARG;
    if (s->nsub > 1) return SPEC_ERR_STATE;   // per-sub-band handles only
    if (fused_failed(s)) return SPEC_ERR_CUDA;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    InputView view{nullptr, (const uint8_t*)d_blocks, 0};
    int rc = 0;
    s->dump = d_out;
    if (s->N1 == 1 || s->r2_single || (s->fused && (s->mode == SPEC_MODE_PFB || !s->use_coef))) {
        rc = run_spectra(s, view, 0, nspec, 0, st);
    } else {
        for (long long b0 = 0; b0 < nspec && !rc; b0 += s->zbatch) {
            const int nb = (int)((nspec - b0 < s->zbatch) ? nspec - b0 : s->zbatch);
            s->dump = d_out + (size_t)b0 * s->N * 2 * s->P;
            rc = run_passA(s, view, b0, nb, st);
        }
    }
    s->dump = nullptr;
    return rc;
}

// ------------------------------------------------------------------ one-shot entry point that allocates nothing
// spec_oneshot_static (include/spec.h): for callers that cannot call cudaMalloc (code under CUDA-graph capture, tight
// serving loops, harnesses that forbid it).  The single-kernel plan (k_engine, nchan <= 4096) needs three pieces of scratch
// besides the caller's input and output: the accumulators in engine position order, the engine's stage twiddles and the
// position -> channel table.  Here they live in ONE file-scope device array of fixed size that every GPU which loads the
// library holds until exit:
//     [0, 64 KiB)        accumulators  float[S][4096] worth of [position][S] sums  (cleared at the start of every call)
//     [64 KiB, 96 KiB)   stage twiddles, at most 4096 float2                        (re-uploaded when nchan changes)
//     [96 KiB, 112 KiB)  position -> channel table, 4096 int                       (re-uploaded when nchan changes)
// In host code the array's NAME is only a host-side stand-in; the device address comes from cudaGetSymbolAddress, taken once
// per device with that device current.  Every call shares the array: calls that overlap on the GPU (two streams) race.
#define SPEC_STATIC_MAX_NCHAN 4096
#define SPEC_STATIC_ACC_BYTES (16 * SPEC_STATIC_MAX_NCHAN)
#define SPEC_STATIC_TW_BYTES (8 * SPEC_STATIC_MAX_NCHAN)
#define SPEC_STATIC_PERM_BYTES (4 * SPEC_STATIC_MAX_NCHAN)
#define SPEC_STATIC_BYTES (SPEC_STATIC_ACC_BYTES + SPEC_STATIC_TW_BYTES + SPEC_STATIC_PERM_BYTES)   // 112 KiB
static __device__ __align__(256) unsigned char g_static_scratch[SPEC_STATIC_BYTES];

struct StaticSetup {
    unsigned char* ptr = nullptr;   // device address of g_static_scratch on this device
    int numSM = 0;
    int nchan = 0;                  // the tables in the array belong to this channel count (0: none yet)
};
static StaticSetup g_static[64];
static std::mutex g_static_mu;
// host staging of the tables (static: nothing is allocated; cudaMemcpyAsync from pageable memory returns once it has
// taken its copy, so the arrays may be rewritten by the next set-up)
static float2 g_static_tw[SPEC_STATIC_MAX_NCHAN];
static int g_static_perm[SPEC_STATIC_MAX_NCHAN];

extern "C" int spec_oneshot_static(const void* d_in, size_t nsamples, int nchan, int ntaps, int npol,
                                   const float* d_coeffs, float* d_out, void* cuda_stream) {
    if (!d_in || !d_out || ((uintptr_t)d_in & 15)) return SPEC_ERR_ARG;
    if (npol != 1 && npol != 2) return SPEC_ERR_ARG;
    if (nchan < 16 || (nchan & (nchan - 1))) return SPEC_ERR_ARG;
    if (nchan > SPEC_STATIC_MAX_NCHAN) {
        snprintf(g_err, sizeof(g_err), "spec_oneshot_static: nchan %d exceeds the static scratch array (at most %d channels, "
                 "%d bytes per GPU); use a spec_create handle for larger transforms", nchan, SPEC_STATIC_MAX_NCHAN, SPEC_STATIC_BYTES);
        return SPEC_ERR_SIZE;
    }
    if (ntaps < 1 || ntaps > 64 || (ntaps > 1 && !d_coeffs)) return SPEC_ERR_ARG;
    if (nsamples % (size_t)nchan) return SPEC_ERR_SIZE;
    const long long nblk = (long long)(nsamples / (size_t)nchan);
    const long long nspec = nblk - (ntaps - 1);
    if (nspec < 1 || nspec > 0x7fffffffll) return SPEC_ERR_SIZE;
    cudaStream_t st = (cudaStream_t)cuda_stream;

    int dev = 0;
    CK(cudaGetDevice(&dev));
    if (dev < 0 || dev >= 64) return SPEC_ERR_ARG;
    std::lock_guard<std::mutex> lk(g_static_mu);
    StaticSetup& su = g_static[dev];
    if (!su.ptr) {   // once per device, with that device current
        unsigned char* p = nullptr;
        CK(cudaGetSymbolAddress((void**)&p, g_static_scratch));
        CK(cudaDeviceGetAttribute(&su.numSM, cudaDevAttrMultiProcessorCount, dev));
        su.ptr = p;
    }
    float* const acc = (float*)su.ptr;
    float2* const tw = (float2*)(su.ptr + SPEC_STATIC_ACC_BYTES);
    int* const perm = (int*)(su.ptr + SPEC_STATIC_ACC_BYTES + SPEC_STATIC_TW_BYTES);
    if (su.nchan != nchan) {   // tables of another channel count (or none): upload this one's, ordered on the caller's stream
        int r[3];
        radices(nchan, r);
        const int LA = nchan / r[0], LB = LA / r[1];
        size_t ntw = 0;
        if (r[1] == 1) g_static_tw[ntw++] = make_float2(1.f, 0.f);
        else {
            for (int q = 1; q < r[0]; q++)
                for (int j = 0; j < LA; j++) {
                    const double a = -2.0 * M_PI * (double)((long)j * q % nchan) / (double)nchan;
                    g_static_tw[ntw++] = make_float2((float)cos(a), (float)sin(a));
                }
            if (r[2] != 1)
                for (int q = 1; q < r[1]; q++)
                    for (int j = 0; j < LB; j++) {
                        const double a = -2.0 * M_PI * (double)((long)j * q % LA) / (double)LA;
                        g_static_tw[ntw++] = make_float2((float)cos(a), (float)sin(a));
                    }
        }
        for (int a = 0; a < nchan; a++) g_static_perm[a] = pos_to_freq(nchan, a);
        su.nchan = 0;
        CK(cudaMemcpyAsync(tw, g_static_tw, ntw * sizeof(float2), cudaMemcpyHostToDevice, st));
        CK(cudaMemcpyAsync(perm, g_static_perm, (size_t)nchan * sizeof(int), cudaMemcpyHostToDevice, st));
        su.nchan = nchan;
    }
    // a handle on the stack that points into the static array: the launch code of the single-kernel plan is reused as it is
    spec_ctx tmp;
    tmp.N = nchan; tmp.T = ntaps; tmp.P = npol; tmp.S = (npol == 2) ? 4 : 1;
    tmp.mode = d_coeffs ? SPEC_MODE_PFB : SPEC_MODE_FFT; tmp.window = SPEC_WINDOW_RECT; tmp.M = (long)nspec;
    tmp.N1 = 1; tmp.N2 = nchan; tmp.numSM = su.numSM;
    tmp.use_coef = d_coeffs != nullptr;
    tmp.d_coef = const_cast<float*>(d_coeffs);
    tmp.d_tw2 = tw; tmp.d_perm = perm; tmp.d_ring = acc; tmp.nring = 1;
    // the array keeps the last call's contents: the sums must start at zero
    CK(cudaMemsetAsync(acc, 0, acc_floats(&tmp) * sizeof(float), st));
    InputView view{nullptr, (const uint8_t*)d_in, 0};
    int rc = run_single(&tmp, view, 0, nspec, 0, st);
    if (rc) return rc;
    k_unpermute<<<cdiv(nchan, 256), 256, 0, st>>>(acc, perm, d_out, nchan, tmp.S, 0, 1);
    CK(cudaGetLastError());
    return (int)nspec;
}

extern "C" int spec_debug_hog(int ms, size_t smem_bytes, void* cuda_stream) {
    if (ms < 0 || ms > 2000 || smem_bytes > 227 * 1024) return SPEC_ERR_ARG;
    int dev = 0, nsm = 0;
    CK(cudaGetDevice(&dev));
    CK(cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev));
    static unsigned* sink = nullptr;
    if (!sink) CK(cudaMalloc(&sink, sizeof(unsigned)));
    CK(cudaFuncSetAttribute(k_debug_hog, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024));
    k_debug_hog<<<nsm, 128, smem_bytes < 512 ? 512 : smem_bytes, (cudaStream_t)cuda_stream>>>((unsigned long long)ms * 1000000ull, sink);
    CK(cudaGetLastError());
    return SPEC_OK;
}

extern "C" int spec_plan_info(const spec_t* s, int* n1, int* n2, char* desc, size_t desc_len) {
    if (!s) return SPEC_ERR_ARG;
    if (s->nsub > 1) {
        char sub[400] = "";
        int rc = spec_plan_info(s->subs[0], n1, n2, sub, sizeof(sub));
        if (desc && desc_len) snprintf(desc, desc_len, "%d sub-bands: k_deinterleave, then per sub-band %s", s->nsub, sub);
        return rc;
    }
    if (n1) *n1 = s->N1;
    if (n2) *n2 = s->N2;
    if (desc && desc_len) {
        const bool pfb = s->mode == SPEC_MODE_PFB;
        int r[3];
        radices(s->N2, r);
        if (s->r2_single)
            snprintf(desc, desc_len, "k_engine<Plan<%d,%d,%d,%d>,FrontRawR2> one launch, two CTAs per spectrum (even / odd channels from "
                     "the whole raw block, first radix-2 layer in the front end): unpack%s+FFT+Stokes+accumulate",
                     s->N2, r[0], r[1], r[2], s->use_coef ? "+window" : "");
        else if (s->N1 == 1)
            snprintf(desc, desc_len, "k_engine<Plan<%d,%d,%d,%d>> single CTA per spectrum: unpack%s+FFT+Stokes+accumulate",
                     s->N2, r[0], r[1], r[2], pfb ? "+FIR" : (s->use_coef ? "+window" : ""));
        else if (s->fused && (pfb || !s->use_coef))
        {
            // (mirrors fused_do's kF2: three-stage row plans; FFT mode, or PFB with 4096-point rows, if the buffers fit)
            const bool f2 = s->N2 >= 512 && (!pfb || (s->N2 == 4096 && s->N1 > 16)) && !(pfb && s->N1 == 128) && !s->tc_stage;
            snprintf(desc, desc_len, "%s<Plan<%d,%d,%d,%d>,%s> persistent four-step %dx%d: unpack%s+FFT+Stokes+accumulate, "
                     "%s, Z ring %d groups x %d spectra",
                     f2 ? "k_fused2" : "k_fused", s->N2, r[0], r[1], r[2], pfb ? "PFB" : "FFT", s->N1, s->N2, pfb ? "+FIR" : "",
                     f2 ? "one producer and one consumer group per CTA, rows prefetched by bulk copy" : "producer and consumer CTAs",
                     s->fRING, s->fGS);
        }
        else
            snprintf(desc, desc_len, "two-launch four-step %dx%d: %s then k_engine<Plan<%d,%d,%d,%d>> pass B, Z batch %d spectra",
                     s->N1, s->N2,
                     (pfb && s->N1 == 16 && s->T == 8) ? "k_passA_pfb16" : (s->d_Y ? "k_fir8 + k_engine pass A" : "k_engine pass A"),
                     s->N2, r[0], r[1], r[2], s->zbatch);
    }
    return SPEC_OK;
}

extern "C" int spec_profile(spec_t* s, int enable) {
    if (!s) return SPEC_ERR_ARG;
    if (s->nsub > 1) {
        for (auto c : s->subs) spec_profile(c, enable);
        return SPEC_OK;
    }
    prof_fold(s);
    s->prof = enable != 0;
    for (int i = 0; i < 4; i++) { s->prof_ms[i] = 0; s->prof_n[i] = 0; }
    return SPEC_OK;
}

extern "C" int spec_profile_read(spec_t* s, double ms[4], long launches[4]) {
    if (!s || !ms || !launches) return SPEC_ERR_ARG;
    if (s->nsub > 1) {
        for (int i = 0; i < 4; i++) { ms[i] = 0; launches[i] = 0; }
        for (auto c : s->subs) {
            double m[4]; long l[4];
            spec_profile_read(c, m, l);
            for (int i = 0; i < 4; i++) { ms[i] += m[i]; launches[i] += l[i]; }
        }
        return SPEC_OK;
    }
    prof_fold(s);
    for (int i = 0; i < 4; i++) { ms[i] = s->prof_ms[i]; launches[i] = s->prof_n[i]; }
    return SPEC_OK;
}
