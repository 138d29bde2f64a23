// fused.cuh — the four-step spectrometer as ONE persistent, self-scheduling kernel (N = 16 * N2).
//
//   A task : unpack + 8-tap FIR (step 3) + 16-point column DFTs + W_N twiddle -> Z ring
//   B job  : Z rows -> N2-point row FFTs (step 4) -> Stokes products -> accumulate
//            (step 5)
//
// The paper runs these as separate kernels around a library FFT, one launch set per FFT invocation
// (PAPER.md:90-95, :116).  Here every CTA of one resident grid is both producer and consumer:
//   * the intermediate Z is a RING of `RING` groups of `GS` spectra that stays in the 126 MB L2;
//     monotonic counters (a_done / b_done per ring slot) order producers and consumers, so a whole
//     spec_process call is one launch however many spectra it holds;
//   * each CTA owns a fixed set of channels (rows k1 of the four-step split) for an interleaved
//     subset of the spectra; their four Stokes sums live in TENSOR MEMORY (tcgen05.ld/st), not in
//     registers, so the FFT runs at 128 registers per thread and four CTAs per SM, and they are
//     added to the HBM accumulator only at accumulation-window boundaries;
//   * thread 0 of every CTA is its scheduler: run my next B job if its spectra are complete in the
//     ring, else claim the next A task if the ring has room, else sleep.  Nothing ever blocks inside
//     a task, dependencies only point to earlier groups, and the grid is exactly the number of CTAs the
//     SMs hold at once (registers, shared memory and TMEM columns all sized for it), so the scheme
//     cannot deadlock.
// Four-step indexing: n = N2*n1 + n2, k = k1 + 16*k2.
#pragma once
#include "engine.cuh"

namespace spk {

struct FusedParams {
    InputView view;        // history ++ input; spectrum j of this launch uses blocks j .. j+T-1
    const float* h;        // T*N coefficients (PFB)
    float4* Z;             // ring: RS spectra of N float4 (Xre, Yre, Xim, Yim), [spectrum][k1][n2]
    const float2* twN;     // W_N^e
    const float2* twL;     // engine stage tables of the N2-point plan
    float* ring;           // accumulator ring (SinkStokesTmem)
    size_t acc_stride;
    int nring;
    int N, N2;
    long long nspec;       // spectra in this launch
    long long c0, M;       // spectra before this launch / per accumulation window
    int GS;                // spectra per group (multiple of the A phase length R)
    int RING;              // groups in the Z ring
    int TPG;               // A tasks (column tiles) per group = N2 / 16
    unsigned long long* dbg;  // optional per-CTA counters (SPEC_FUSED_DEBUG): 8 words per CTA
    unsigned* flags;       // [0] next A task, [1 .. RING] a_done, [1+RING .. 2*RING] b_done (zeroed per launch)
};

__device__ __forceinline__ unsigned ld_acquire_u32(const unsigned* p) {
    unsigned v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ unsigned ld_relaxed_u32(const unsigned* p) {
    unsigned v;
    asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}

// ---------------------------------------------------------------- A task
// C = 16 adjacent columns n2 (all 16 rows n1: 256 filter branches), the GS spectra of one group,
// R = NT/16 spectra per phase.  FIR phase: each thread owns 16/R*... branches and slides an 8-sample
// register window over R+7 blocks; FFT phase: each thread owns one (spectrum, column) pair.
template <int NT, int MODE_PFB>
__device__ __forceinline__ void fused_task_A(const FusedParams& p, float4* ysm, long long g, int tile) {
    constexpr int C = 16, R = NT / C, T = 8;
    constexpr int BPT = 16 * C / NT;  // branches per thread in the FIR phase
    const int tid = threadIdx.x;
    const int N = p.N, N2 = p.N2;
    const int n2_0 = tile * C;
    const long long mg = g * p.GS;                                    // first spectrum of the group
    const int nsp = (int)((p.nspec - mg < p.GS) ? p.nspec - mg : p.GS);  // valid spectra in it
    const int fr = tid / C, fc = tid % C;
    const int n2 = n2_0 + fc;
    float4* const zg = p.Z + (size_t)((mg % ((long long)p.RING * p.GS))) * N + n2;

    float2 tw[16];
#pragma unroll
    for (int k = 1; k < 16; k++) tw[k] = __ldg(p.twN + (size_t)n2 * k);

    if (MODE_PFB) {
        float hc[BPT][T];
        int nbr[BPT];
#pragma unroll
        for (int i = 0; i < BPT; i++) {
            const int beta = tid + NT * i;
            nbr[i] = (beta / C) * N2 + n2_0 + (beta % C);
#pragma unroll
            for (int t = 0; t < T; t++) hc[i][t] = __ldg(p.h + (size_t)t * N + nbr[i]);
        }
        for (int j0 = 0; j0 < nsp; j0 += R) {
            // ---------------- FIR phase: all raw words first (one L2 latency per phase)
            const int qmax = nsp - 1 - j0 + (T - 1);  // last valid block of this phase (ragged tail)
            uint32_t raw[BPT][R + T - 1];
            const bool in_input = (mg + j0 >= p.view.nhist);
#pragma unroll
            for (int i = 0; i < BPT; i++) {
                if (in_input) {
                    const uint32_t* base = (const uint32_t*)p.view.in + (size_t)(mg + j0 - p.view.nhist) * N + nbr[i];
#pragma unroll
                    for (int q = 0; q < R + T - 1; q++) raw[i][q] = __ldg(base + (size_t)(q < qmax ? q : qmax) * N);
                } else {
#pragma unroll
                    for (int q = 0; q < R + T - 1; q++)
                        raw[i][q] = fetch_raw<2>(p.view, mg + j0 + (q < qmax ? q : qmax), nbr[i], N);
                }
            }
#pragma unroll
            for (int i = 0; i < BPT; i++) {
                const int beta = tid + NT * i;
                const int n1 = beta / C, c = beta % C;
                cpx x[T];
#pragma unroll
                for (int t = 0; t < T - 1; t++) x[t] = unpack_cpx<2>(raw[i][t]);
#pragma unroll
                for (int r = 0; r < R; r++) {
                    x[(r + T - 1) % T] = unpack_cpx<2>(raw[i][r + T - 1]);
                    u64 re = 0ull, im = 0ull;
#pragma unroll
                    for (int t = 0; t < T; t++) {
                        re = fma2(x[(r + t) % T].re, bc(hc[i][t]), re);
                        im = fma2(x[(r + t) % T].im, bc(hc[i][t]), im);
                    }
                    ysm[(r * 16 + n1) * C + c] = cpx_to_f4({re, im});
                }
            }
            __syncthreads();
            // ---------------- column FFT phase
            if (j0 + fr < nsp) {
                cpx v[16];
#pragma unroll
                for (int n1 = 0; n1 < 16; n1++) v[n1] = f4_to_cpx(ysm[(fr * 16 + n1) * C + fc]);
                dft<16>(v);
                float4* zp = zg + (size_t)(j0 + fr) * N;
                zp[0] = cpx_to_f4(v[0]);
#pragma unroll
                for (int k = 1; k < 16; k++) zp[(size_t)k * N2] = cpx_to_f4(cmul(v[k], tw[k].x, tw[k].y));
            }
            __syncthreads();
        }
    } else {
        // direct-FFT mode: no pre-filter, the 16 samples of a column go straight from
        // global memory through the unpack into the butterfly
        for (int j0 = 0; j0 < nsp; j0 += R) {
            if (j0 + fr < nsp) {
                const uint32_t* base = (const uint32_t*)p.view.in + (size_t)(mg + j0 + fr) * N + n2;
                uint32_t raw[16];
#pragma unroll
                for (int n1 = 0; n1 < 16; n1++) raw[n1] = __ldg(base + (size_t)n1 * N2);
                cpx v[16];
#pragma unroll
                for (int n1 = 0; n1 < 16; n1++) v[n1] = unpack_cpx<2>(raw[n1]);
                dft<16>(v);
                float4* zp = zg + (size_t)(j0 + fr) * N;
                zp[0] = cpx_to_f4(v[0]);
#pragma unroll
                for (int k = 1; k < 16; k++) zp[(size_t)k * N2] = cpx_to_f4(cmul(v[k], tw[k].x, tw[k].y));
            }
        }
        __syncthreads();
    }
}

// ---------------------------------------------------------------- the kernel
template <class PL, int NT, int MODE_PFB>
__global__ void __launch_bounds__(NT, 512 / NT)
k_fused(const FusedParams p) {
    constexpr int L = PL::L, RA = PL::RA, RB = PL::RB, RC = PL::RC, NST = PL::NST;
    constexpr int LA = PL::LA, LB = PL::LB, NTS = PL::NTS;
    constexpr int G = NT / NTS;                     // rows per B job
    constexpr int RGN = (G >= 16) ? 1 : 16 / G;     // row groups per spectrum
    constexpr int SPJ = (G >= 16) ? G / 16 : 1;     // spectra per B job
    constexpr int TCOLS = (NT > 128) ? 128 : 64;
    static_assert(NST >= 2 && PL::RLAST == 16 && G * L * 16 == NT * 256, "row plan");
    extern __shared__ float4 smem[];                // G*L float4: B exchange buffer / A FIR hand-off
    __shared__ int s_ctl[2][4];
    __shared__ uint32_t s_tmem;

    const int tid = threadIdx.x;
    const int slot = tid / NTS, t = tid % NTS;
    unsigned* const a_next = p.flags;
    unsigned* const a_done = p.flags + 1;
    unsigned* const b_done = p.flags + 1 + p.RING;

    // B ownership: row group rg of every (y + i*ny)-th job
    const int rg = blockIdx.x % RGN;
    const int y = blockIdx.x / RGN;
    const int ny = gridDim.x / RGN;
    const long long njobs_all = (p.nspec + SPJ - 1) / SPJ;
    const long long nbj = (y < ny && y < njobs_all) ? (njobs_all - y + ny - 1) / ny : 0;  // my B jobs
    const int row = (G >= 16) ? (slot % 16) : (rg * G + slot);
    const int sub = (G >= 16) ? (slot / 16) : 0;    // spectrum of the job this slot works on

    auto addr = [&](int q) -> int { return slot * L + (q ^ ((q / 16) & 7)); };

    const uint32_t tmem_base = tmem_alloc_cta<TCOLS>(&s_tmem);
    SinkStokesTmem sink{p.ring, p.acc_stride, p.nring, L, 1};
    SinkStokesTmem::State st;
    sink.init(st, tmem_base);
    sink.begin(st);
    long long wcur = -1;   // accumulation window the TMEM sums belong to (-1: none yet)

    long long bi = 0;      // my next B job (kept by every thread)
    // scheduler state (thread 0)
    long long ready_g = -1;   // a group known to be complete in the ring
    long long freed_g = -1;   // a group known to be fully consumed
    long long pend_a = -1;    // claimed A task waiting for its ring slot
    bool a_exhausted = false;
    const long long ngroups = (p.nspec + p.GS - 1) / p.GS;
    const long long natasks = ngroups * p.TPG;

    unsigned long long d_idle = 0, d_na = 0, d_nb = 0, d_ta = 0, d_tb = 0, d_ti = 0, d_t0 = clock64(), d_last = d_t0;
    for (int it = 0;; it++) {
        int* ctl = s_ctl[it & 1];
        if (tid == 0) {
            int type = 0;  // 0 idle, 1 B job, 2 A task, 3 exit
            long long atask = 0;
            if (bi < nbj) {
                const long long s0 = (y + bi * ny) * SPJ;
                long long s1 = s0 + SPJ - 1;
                if (s1 > p.nspec - 1) s1 = p.nspec - 1;
                const long long g = s1 / p.GS;
                if (g <= ready_g) type = 1;
                else if (ld_acquire_u32(a_done + g % p.RING) >= (unsigned)((g / p.RING + 1) * p.TPG)) {
                    // groups complete in any order, but my jobs ask about non-decreasing g, and a group
                    // can only be overwritten after I have consumed my rows of it
                    ready_g = g;
                    type = 1;
                }
            }
            if (type == 0) {
                // claim the next A task unconditionally (a failed compare-and-swap would serialise the
                // whole grid), then hold it until its ring slot is free; meanwhile keep serving B jobs
                if (pend_a < 0 && !a_exhausted) {
                    const unsigned a = atomicAdd(a_next, 1u);
                    if ((long long)a >= natasks) a_exhausted = true;
                    else pend_a = a;
                }
                if (pend_a >= 0) {
                    const long long g = pend_a / p.TPG;
                    if (g < p.RING || g - p.RING <= freed_g ||
                        ld_acquire_u32(b_done + g % p.RING) >= (unsigned)((g / p.RING) * p.GS * 16)) {
                        if (g >= p.RING) freed_g = g - p.RING;
                        type = 2;
                        atask = pend_a;
                        pend_a = -1;
                    }
                }
            }
            if (type == 0 && bi >= nbj && a_exhausted && pend_a < 0) type = 3;
            ctl[0] = type;
            ctl[1] = (int)atask;
        }
        __syncthreads();
        const int type = ctl[0];
        if (type == 3) break;
        if (type == 0) {
            __nanosleep(100);
            if (p.dbg && tid == 0) { const unsigned long long c = clock64(); d_ti += c - d_last; d_last = c; d_idle++; }
            continue;
        }
        if (type == 2) {
            const long long a = ctl[1];
            const long long g = a / p.TPG;
            fused_task_A<NT, MODE_PFB>(p, smem, g, (int)(a % p.TPG));   // ends with a __syncthreads
            if (tid == 0) {
                __threadfence();
                atomicAdd(a_done + g % p.RING, 1u);
            }
            if (p.dbg && tid == 0) { const unsigned long long c = clock64(); d_ta += c - d_last; d_last = c; d_na++; }
            continue;
        }
        // ---------------- B job bi
        const long long s0 = (y + bi * ny) * SPJ;
        const long long m = s0 + sub;
        const bool active = m < p.nspec;
        if (active) {
            const long long w = (p.c0 + m) / p.M;
            if (w != wcur) {   // warp-uniform: a warp never straddles spectra
                if (wcur >= 0) { sink.flush(st, row, t, wcur); sink.begin(st); }
                wcur = w;
            }
        }
        const float4* zrow = p.Z + (size_t)(m % ((long long)p.RING * p.GS)) * p.N + (size_t)row * L;
        // stage a: rows of Z straight from L2 (ld.global.cg: the ring is rewritten by other SMs)
        if (active) {
#pragma unroll
            for (int u = 0; u < 16 / RA; u++) {
                const int ja = t + NTS * u;
                cpx v[RA];
#pragma unroll
                for (int r = 0; r < RA; r++) v[r] = f4_to_cpx(__ldcg(zrow + ja + r * LA));
                dft<RA>(v);
                smem[addr(ja)] = cpx_to_f4(v[0]);
#pragma unroll
                for (int q = 1; q < RA; q++) {
                    const float2 w = __ldg(p.twL + (q - 1) * LA + ja);
                    smem[addr(ja + q * LA)] = cpx_to_f4(cmul(v[q], w.x, w.y));
                }
            }
        }
        __syncthreads();
        if (tid == 0) {   // my rows of this job are consumed: let the producers reuse the ring slot
            long long s1 = s0 + SPJ;
            if (s1 > p.nspec) s1 = p.nspec;
            const unsigned rows = (G >= 16) ? (unsigned)(16 * (s1 - s0)) : (unsigned)G;
            __threadfence();
            atomicAdd(b_done + (s0 / p.GS) % p.RING, rows);
        }
        bi++;
        if (active) {
#pragma unroll
            for (int u = 0; u < 16 / RB; u++) {
                const int i = t + NTS * u;
                const int qa = i / LB, jb = i % LB;
                const int base = qa * LA + jb;
                cpx v[RB];
#pragma unroll
                for (int r = 0; r < RB; r++) v[r] = f4_to_cpx(smem[addr(base + r * LB)]);
                dft<RB>(v);
                if (NST == 2) {
                    sink.put16(st, m, 0, i, i, RA, v);
                } else {
                    smem[addr(base)] = cpx_to_f4(v[0]);
#pragma unroll
                    for (int q = 1; q < RB; q++) {
                        const float2 w = __ldg(p.twL + (RA - 1) * LA + (q - 1) * LB + jb);
                        smem[addr(base + q * LB)] = cpx_to_f4(cmul(v[q], w.x, w.y));
                    }
                }
            }
        }
        if (NST == 3) {
            __syncthreads();
            if (active) {
                cpx v[RC];
#pragma unroll
                for (int r = 0; r < RC; r++) v[r] = f4_to_cpx(smem[addr(t * RC + r)]);
                dft<RC>(v);
                sink.put16(st, m, 0, t, 0, 1, v);
            }
        }
        // the scheduler's barrier at the top of the next iteration also protects the exchange buffer
        if (p.dbg && tid == 0) { const unsigned long long c = clock64(); d_tb += c - d_last; d_last = c; d_nb++; }
    }
    if (p.dbg && tid == 0) {
        unsigned long long* d = p.dbg + (size_t)blockIdx.x * 8;
        d[0] = d_idle; d[1] = d_na; d[2] = d_nb; d[3] = d_ti; d[4] = d_ta; d[5] = d_tb; d[6] = clock64() - d_t0; d[7] = d_t0;
    }
    if (wcur >= 0) sink.flush(st, row, t, wcur);
    tmem_free_cta<TCOLS>(tmem_base);
}

}  // namespace spk
