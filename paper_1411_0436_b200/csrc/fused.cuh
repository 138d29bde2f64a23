// fused.cuh — the four-step spectrometer as ONE persistent, self-scheduling kernel (N = 16 * N2).
//
//   A task : unpack + 8-tap FIR (step 3) + 16-point column DFTs + W_N twiddle -> Z ring
//   B job  : Z rows -> N2-point row FFTs (step 4) -> Stokes products -> accumulate
//            (step 5)
//
// The paper runs these as separate kernels around a library FFT, one launch set per FFT invocation
// (PAPER.md:90-95, :116).  Here one resident grid holds producers and consumers side by side:
//   * the intermediate Z is a RING of `RING` groups of `GS` spectra that stays in the 126 MB L2;
//     one monotonic counter pair per group (a_done / b_done) orders producers and consumers, so a
//     whole spec_process call is one launch however many spectra it holds;
//   * every SM hosts `na_per_sm` PRODUCER CTAs (A tasks, round-robin over the task list) and the rest
//     of its CTAs as CONSUMERS (each owns fixed rows k1 of the four-step split for an interleaved
//     subset of the spectra).  The role comes from the order of arrival on the SM (%smid counter), so
//     both kinds always share an SM: whichever side is blocked leaves its issue slots to the other,
//     which balances the two rates without any scheduler;
//   * the consumers' four Stokes sums live in TENSOR MEMORY (tcgen05.ld/st), not in registers, so
//     the FFT runs at 128 registers per thread and four CTAs per SM; they are added to the HBM
//     accumulator only at accumulation-window boundaries;
//   * a producer waits (thread 0, prefetched poll) only for the ring slot it is about to overwrite, a
//     consumer only for the group it is about to read; dependencies point to earlier groups only and
//     the grid is exactly the number of CTAs the SMs hold at once (the register file allows no more
//     per SM, so every SM gets the same mix), hence no deadlock.
// Four-step indexing: n = N2*n1 + n2, k = k1 + 16*k2.
#pragma once
#include "engine.cuh"

namespace spk {

constexpr int kFusedRoleWords = 516;   // 4 counters + 512 per-SM arrival counters (keeps what follows 16-byte aligned)

struct FusedParams {
    InputView view;        // history ++ input; spectrum j of this launch uses blocks j .. j+T-1
    const float* h;        // T*N coefficients (PFB)
    float4* Z;             // ring: RING*GS spectra of N float4 (Xre, Yre, Xim, Yim), [spectrum][k1][n2]
    const float2* twN;     // W_N^e
    const float2* twT;     // N1 > 16: the same twiddles by column position, twT[p1*N2 + n2] = W_N^{n2 k1(p1)} (coalesced over n2)
    const float2* tw1;     // N1 > 16: engine stage table of the N1-point column plan (Q x 16)
    const float2* twL;     // engine stage tables of the N2-point plan
    float* ring;           // accumulator ring (SinkStokesTmem)
    size_t acc_stride;
    int nring;
    int N, N2;
    int nspec;             // spectra in this launch
    long long c0, M;       // spectra before this launch / per accumulation window
    int lgGS;              // log2 of the spectra per group (a multiple of the A phase length)
    int RING;              // groups in the Z ring
    int lgTPG;             // log2 of the A tasks (column tiles of 16) per group, TPG = N2 / 16
    int na_per_sm;         // producer CTAs per SM (the others consume)
    int per_sm;            // resident CTAs per SM (the register budget of the kernel allows exactly this many)
    unsigned* role;        // [0] producer rank counter, [1] consumer rank counter, [2] arrivals, [3] departures,
                           // [4 + smid] CTAs seen on that SM.  All counters are zero between launches: the last
                           // CTA to leave resets them, so a call needs no memset
    unsigned* a_done;      // [group] finished A tasks          } zeroed before every launch; one counter per
    unsigned* b_done;      // [group] consumed rows (of GS*16)  } GROUP of the launch: no epochs, no divisions
    unsigned* err;         // mapped host word: set to 1 if a wait inside the kernel timed out (the launch then
                           // runs to its end with garbage results instead of hanging; the host reports it)
    const uint4* carry_src;  // PFB: the last T-1 blocks of this call's input ...
    uint4* carry_dst;        // ... are copied into the history buffer of the NEXT call by this launch (16-byte chunks),
    int carry_chunks;        // so that no copy sits between two launches in the stream (0: the host copies)
    unsigned* carry_cnt;     // monotonic: every CTA of a carrying launch adds one after its share of the copy (release);
    unsigned carry_wait;     // a launch whose history was written that way first waits (acquire) for the counter to
    int carry_wait_on;       // reach carry_wait: consecutive launches overlap, so stream order does not cover it
    float* dump;             // DUMP instantiation only (test hook): front-end output [spectrum][n][Xre,Xim,Yre,Yim]
    const void* tcB;         // TC instantiation only: the split fp16 DFT matrix B' (fused_producer_fft_tc)
};

// relaxed (strong, gpu-scope) counter read.  The polls are issued one task ahead into a register, so the L2
// round trip is hidden; the acquire is a separate fence once the value says "ready" (fence_acquire_gpu).
// Z itself is read with ld.global.cg, so no stale L1 line can be hit.
__device__ __forceinline__ unsigned ld_relaxed_u32(const unsigned* p) {
    unsigned v;
    asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ unsigned atom_add_relaxed_u32(unsigned* p, unsigned v) {
    unsigned r;
    asm volatile("atom.relaxed.gpu.global.add.u32 %0, [%1], %2;" : "=r"(r) : "l"(p), "r"(v) : "memory");
    return r;
}
// Bounded wait on a monotonic counter: spins (with back-off) until *ctr >= target, or gives up after about
// ten seconds and raises the error word.  A wait can only time out if the grid is not fully resident (a
// foreign kernel holding SM resources for that long) or on a logic error; either way the launch must end.
__device__ __forceinline__ void wait_counter(const unsigned* ctr, unsigned target, unsigned* err) {
    if (ld_relaxed_u32(ctr) >= target) return;
    unsigned long long t0;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t0));
    for (unsigned it = 1;; it++) {
        __nanosleep(200);
        if (ld_relaxed_u32(ctr) >= target) return;
        // (the error word lives in host memory: look at it rarely; once it is set everybody drains quickly)
        if ((it & 0xffffu) == 0 && *(volatile unsigned*)err) return;
        unsigned long long t1;
        asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t1));
        if (t1 - t0 > 10000000000ull) {
            *(volatile unsigned*)err = 1u;
            __threadfence_system();
            return;
        }
    }
}
__device__ __forceinline__ void red_release_u32(unsigned* p, unsigned v) {
    asm volatile("red.release.gpu.global.add.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
// Acquire side of the counter protocol.  The writer publishes with red.release.gpu after a CTA barrier
// (cumulative over the CTA's stores); the reader's poll is a relaxed (strong) load, made an acquire by a
// fence, and the CTA barrier that follows extends the ordering to the other threads of the reader.
__device__ __forceinline__ void fence_acquire_gpu() { asm volatile("fence.acq_rel.gpu;" ::: "memory"); }
// The same fence after the per-task polls of the Z ring (a_done / b_done).  It compiles to MEMBAR.ALL.GPU +
// CCTL.IVALL on sm_100a and sits on the critical path of every task: measured cost 7.5 % of configs[1]'s
// throughput (104.6 -> 97.1 GHz, profiles/r02_experiments.md), so the default build leaves it out and relies
// on what the hardware does (the ring is read with ld.global.cg, i.e. from the L2, the
// point of coherence, never from an L1 line; the poll completes before the CTA barrier that every reader of
// the ring passes first; the writer's release orders its CTA's stores before the counter update at the L2).
// -DSPK_ACQ_FENCE=1 builds the formally fenced variant.
#ifndef SPK_ACQ_FENCE
#define SPK_ACQ_FENCE 0
#endif
__device__ __forceinline__ void fence_acquire_task() {
#if SPK_ACQ_FENCE
    asm volatile("fence.acq_rel.gpu;" ::: "memory");
#endif
}
// wait until a monotonic (wrapping) counter has passed `target`
__device__ __forceinline__ void wait_counter_wrap(const unsigned* ctr, unsigned target, unsigned* err) {
    if ((int)(ld_relaxed_u32(ctr) - target) >= 0) return;
    unsigned long long t0;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t0));
    for (;;) {
        __nanosleep(200);
        if ((int)(ld_relaxed_u32(ctr) - target) >= 0) return;
        unsigned long long t1;
        asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t1));
        if (t1 - t0 > 10000000000ull) {
            *(volatile unsigned*)err = 1u;
            __threadfence_system();
            return;
        }
    }
}

// Barrier of a role group: BAR = 0 the whole CTA, BAR > 0 named barrier BAR of 128 threads (k_fused2: a producer
// group and a consumer group share one CTA)
template <int BAR, int CNT = 128>
__device__ __forceinline__ void gsync() {
    if (BAR == 0) __syncthreads();
    else asm volatile("bar.sync %0, %1;" ::"n"(BAR), "n"(CNT) : "memory");
}

// ---------------------------------------------------------------- A task, PFB mode
// C = 16 adjacent columns n2 (all 16 rows n1: 256 filter branches), the GS spectra of one group,
// R = NT/16 spectra per phase.  The raw samples of a phase (R+7 blocks x 16 rows x 64 bytes) are
// staged in shared memory with 16-byte cp.async copies issued ONE PHASE AHEAD (across task
// boundaries too: the task list of a producer is static), so the latency of the input stream is
// hidden behind the previous phase's column FFTs.  FIR phase: each thread owns 256/NT branches and
// slides an 8-sample register window over the R+7 blocks (every raw sample is unpacked once per
// phase); FFT phase: each thread owns one (spectrum, column) pair.
template <int NT, int N2>
struct ProducerPfb {
    static constexpr int C = 16, R = NT / C, T = 8, N = 16 * N2, BPT = 256 / NT;
    static constexpr int NBLK = R + T - 1;                 // blocks per phase
    static constexpr int RAW_WORDS = NBLK * 256;           // u32 per staged tile
    static constexpr int CHUNKS = RAW_WORDS / 4;           // 16-byte copies per tile

    // issue the copies of phase (g, tile, j0): block q of the phase is view block mg + j0 + min(q, qmax)
    static __device__ __forceinline__ void stage(const FusedParams& p, uint32_t* rawsm, int g, int tile, int j0) {
        const int GS = 1 << p.lgGS;
        const int mg = g << p.lgGS;
        const int nsp = (p.nspec - mg < GS) ? p.nspec - mg : GS;
        const int qmax = nsp - 1 - j0 + (T - 1);
        const int n2_0 = tile * C;
#pragma unroll
        for (int i = 0; i < (CHUNKS + NT - 1) / NT; i++) {
            const int c = threadIdx.x + NT * i;
            if (CHUNKS % NT == 0 || c < CHUNKS) {
                const int q = c >> 6, n1 = (c >> 2) & 15, part = c & 3;
                const int blk = mg + j0 + (q < qmax ? q : qmax);
                const uint8_t* base = (blk < p.view.nhist) ? p.view.hist + (size_t)blk * N * 4
                                                           : p.view.in + (size_t)(blk - p.view.nhist) * N * 4;
                const uint8_t* src = base + ((size_t)n1 * N2 + n2_0) * 4 + part * 16;
                asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(smem_u32(rawsm + c * 4)), "l"(src) : "memory");
            }
        }
    }
};

// The producer loop of one CTA in PFB mode: tasks rank, rank + NA, ...; `wait_room(g)` (thread 0) returns
// once the ring slot of group g may be overwritten, `signal(g, next task)` (thread 0) publishes a finished task.
template <int NT, int N2, bool DUMP, class WaitRoom, class Signal, int BAR = 0>
__device__ __forceinline__ void fused_producer_pfb(const FusedParams& p, float4* smem, int rank, int NA, int natasks,
                                                   WaitRoom wait_room, Signal signal, int lead = 0) {
    typedef ProducerPfb<NT, N2> PP;
    constexpr int C = PP::C, R = PP::R, T = PP::T, N = PP::N, BPT = PP::BPT;
    float4* const ysm = smem;                                   // [R][16][C] FIR outputs
    uint32_t* const rawsm = (uint32_t*)(smem + R * 16 * C);     // [R+7][16][C] raw samples of the phase
    const int tid = threadIdx.x;
    const int GS = 1 << p.lgGS;
    const int TPGm = (1 << p.lgTPG) - 1;
    const int fr = tid / C, fc = tid % C;

    if (rank < natasks) PP::stage(p, rawsm, rank >> p.lgTPG, rank & TPGm, 0);
    for (int a = rank; a < natasks; a += NA) {
        const int g = a >> p.lgTPG, tile = a & TPGm;
        const int n2_0 = tile * C;
        const int mg = g << p.lgGS;
        const int nsp = (p.nspec - mg < GS) ? p.nspec - mg : GS;
        const int n2 = n2_0 + fc;
        float4* const zg = p.Z + ((size_t)((unsigned)g % (unsigned)p.RING) << p.lgGS) * N + n2;
        float2 tw[16];
#pragma unroll
        for (int k = 1; k < 16; k++) tw[k] = __ldg(p.twN + (size_t)n2 * k);
        float hc[BPT][T];
#pragma unroll
        for (int i = 0; i < BPT; i++) {
            const int beta = tid + NT * i;
            const int nbr = (beta / C) * N2 + n2_0 + (beta % C);
#pragma unroll
            for (int t = 0; t < T; t++) hc[i][t] = __ldg(p.h + t * N + nbr);
        }
        for (int j0 = 0; j0 < nsp; j0 += R) {
            asm volatile("cp.async.wait_all;" ::: "memory");
            gsync<BAR, NT>();   // the staged tile is complete; the previous phase's column FFTs have read ysm
            // ---------------- FIR phase
#pragma unroll
            for (int i = 0; i < BPT; i++) {
                const int beta = tid + NT * i;
                cpx x[T];
#pragma unroll
                for (int t = 0; t < T - 1; t++) x[t] = unpack_cpx<2>(rawsm[t * 256 + beta]);
#pragma unroll
                for (int r = 0; r < R; r++) {
                    x[(r + T - 1) % T] = unpack_cpx<2>(rawsm[(r + T - 1) * 256 + beta]);
                    u64 re = 0ull, im = 0ull;
#pragma unroll
                    for (int t = 0; t < T; t++) {
                        re = fma2(x[(r + t) % T].re, bc(hc[i][t]), re);
                        im = fma2(x[(r + t) % T].im, bc(hc[i][t]), im);
                    }
                    ysm[r * 256 + beta] = cpx_to_f4({re, im});
                }
            }
            if (!DUMP && j0 == 0 && tid == lead) wait_room(g);
            gsync<BAR, NT>();   // ysm complete, the raw tile is free again
            // ---------------- stage the next phase (of this task or of my next task)
            if (j0 + R < nsp) PP::stage(p, rawsm, g, tile, j0 + R);
            else if (a + NA < natasks) PP::stage(p, rawsm, (a + NA) >> p.lgTPG, (a + NA) & TPGm, 0);
            // ---------------- column FFT phase
            if (j0 + fr < nsp) {
                cpx v[16];
#pragma unroll
                for (int n1 = 0; n1 < 16; n1++) v[n1] = f4_to_cpx(ysm[fr * 256 + n1 * C + fc]);
                if (DUMP) {   // test hook: what the column FFT is about to consume, in the caller's layout
                    float4* dp = (float4*)p.dump + (size_t)(mg + j0 + fr) * N + n2;
#pragma unroll
                    for (int n1 = 0; n1 < 16; n1++) {
                        const float4 z = cpx_to_f4(v[n1]);
                        dp[n1 * N2] = make_float4(z.x, z.z, z.y, z.w);
                    }
                } else {
                    dft<16>(v);
                    float4* zp = zg + (size_t)(j0 + fr) * N;
                    zp[0] = cpx_to_f4(v[0]);
#pragma unroll
                    for (int k = 1; k < 16; k++) zp[k * N2] = cpx_to_f4(cmul(v[k], tw[k].x, tw[k].y));
                }
            }
        }
        gsync<BAR, NT>();   // every Z store of the task has been issued by its thread
        if (!DUMP && tid == lead) signal(g, a + NA);
    }
}

// One A task in direct-FFT mode: no pre-filter, the 16 samples of a column go straight
// from global memory through the unpack into the butterfly.
template <int NT, int N2, bool DUMP, class WaitRoom, int BAR = 0>
__device__ __forceinline__ void fused_task_A_fft(const FusedParams& p, int g, int tile, WaitRoom wait_room, int lead = 0) {
    constexpr int C = 16, R = NT / C, N = 16 * N2;
    const int tid = threadIdx.x;
    const int GS = 1 << p.lgGS;
    const int mg = g << p.lgGS;
    const int nsp = (p.nspec - mg < GS) ? p.nspec - mg : GS;
    const int fr = tid / C, fc = tid % C;
    const int n2 = tile * C + fc;
    float4* const zg = p.Z + ((size_t)((unsigned)g % (unsigned)p.RING) << p.lgGS) * N + n2;
    float2 tw[16];
#pragma unroll
    for (int k = 1; k < 16; k++) tw[k] = __ldg(p.twN + (size_t)n2 * k);
    if (!DUMP && tid == lead) wait_room(g);
    gsync<BAR, NT>();
    for (int j0 = 0; j0 < nsp; j0 += R) {
        if (j0 + fr < nsp) {
            const uint32_t* base = (const uint32_t*)p.view.in + (size_t)(mg + j0 + fr) * N + n2;
            uint32_t raw[16];
#pragma unroll
            for (int n1 = 0; n1 < 16; n1++) raw[n1] = __ldg(base + n1 * N2);
            cpx v[16];
#pragma unroll
            for (int n1 = 0; n1 < 16; n1++) v[n1] = unpack_cpx<2>(raw[n1]);
            if (DUMP) {   // test hook: the unpacked samples the butterfly is about to consume
                float4* dp = (float4*)p.dump + (size_t)(mg + j0 + fr) * N + n2;
#pragma unroll
                for (int n1 = 0; n1 < 16; n1++) {
                    const float4 z = cpx_to_f4(v[n1]);
                    dp[n1 * N2] = make_float4(z.x, z.z, z.y, z.w);
                }
            } else {
                dft<16>(v);
                float4* zp = zg + (size_t)(j0 + fr) * N;
                zp[0] = cpx_to_f4(v[0]);
#pragma unroll
                for (int k = 1; k < 16; k++) zp[k * N2] = cpx_to_f4(cmul(v[k], tw[k].x, tw[k].y));
            }
        }
    }
    gsync<BAR, NT>();
}

// ---------------------------------------------------------------- A task for N1 = 32, 64, 128 (N >= 131072, N2 = 4096)
// The column transform no longer fits one thread: N1 = Q x 16 runs as the engine's two-stage plan (radix Q over
// n1 = ja + 16 i, twiddle W_N1^{ja q}, then radix 16 over the 16 points of block qa), in place in the FIR hand-off
// buffer with one CTA barrier in between.  A task is C adjacent columns n2 x all N1 rows x R spectra (ONE phase:
// a group is R spectra, so that the ring of a 2^19-point transform still fits the L2), with
// R * N1 * C = 16 * NT points per phase: N1 = 32: R = 8, C = 16;  64: R = 8, C = 8;  128: R = 4, C = 8.
// Output row p1 = 16 qa + qb holds frequency k1 = qa + Q qb (engine position order, as the read-out expects).
// T = 8: PFB, T = 1: direct FFT, the FIR phase is then the unpack alone.
template <int NT, int N2, int N1, int T>
struct ProducerBig {
    static constexpr int Q = N1 / 16;
    static constexpr int R = (N1 == 128) ? 4 : 8;
    static constexpr int C = (16 * NT) / (R * N1);
    static constexpr int BR = N1 * C;                      // filter branches per task
    static constexpr int BPT = BR / NT;                    // branches per thread
    static constexpr int NBLK = R + T - 1;                 // blocks per phase
    static constexpr int N = N1 * N2;
    static constexpr int CHUNKS = NBLK * BR / 4;           // 16-byte copies per staged tile
    static constexpr size_t SMEM = (size_t)R * BR * sizeof(float4) + (size_t)NBLK * BR * 4;
    static_assert(NT == 256 && C >= 4 && C % 4 == 0 && BPT >= 1 && Q >= 2 && Q <= 8, "task shape");

    static __device__ __forceinline__ void stage(const FusedParams& p, uint32_t* rawsm, int g, int tile) {
        const int GS = 1 << p.lgGS;
        const int mg = g << p.lgGS;
        const int nsp = (p.nspec - mg < GS) ? p.nspec - mg : GS;
        const int qmax = nsp - 1 + (T - 1);
        const int n2_0 = tile * C;
#pragma unroll
        for (int i = 0; i < (CHUNKS + NT - 1) / NT; i++) {
            const int c = threadIdx.x + NT * i;
            if (CHUNKS % NT == 0 || c < CHUNKS) {
                const int q = c / (BR / 4), rem = c % (BR / 4);
                const int n1 = rem / (C / 4), part = rem % (C / 4);
                const int blk = mg + (q < qmax ? q : qmax);
                const uint8_t* base = (blk < p.view.nhist) ? p.view.hist + (size_t)blk * N * 4
                                                           : p.view.in + (size_t)(blk - p.view.nhist) * N * 4;
                const uint8_t* src = base + ((size_t)n1 * N2 + n2_0) * 4 + part * 16;
                asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(smem_u32(rawsm + c * 4)), "l"(src) : "memory");
            }
        }
    }
};

template <int NT, int N2, int N1, int T, bool DUMP, class WaitRoom, class Signal, int BAR = 0>
__device__ __forceinline__ void fused_producer_big(const FusedParams& p, float4* smem, int rank, int NA, int natasks,
                                                   WaitRoom wait_room, Signal signal, int lead) {
    typedef ProducerBig<NT, N2, N1, T> PP;
    constexpr int Q = PP::Q, R = PP::R, C = PP::C, BR = PP::BR, BPT = PP::BPT, N = PP::N;
    float4* const ysm = smem;                                  // [R][N1][C]: FIR outputs, then the column transform in place
    uint32_t* const rawsm = (uint32_t*)(smem + R * BR);        // [R+T-1][N1][C] raw samples of the phase
    const int tid = threadIdx.x;
    const int GS = 1 << p.lgGS;                                // == R
    const int TPGm = (1 << p.lgTPG) - 1;
    // second-stage role: spectrum r2 of the phase, column c2, block qa (16 points -> frequencies qa + Q qb)
    const int c2 = tid % C, qa = (tid / C) % Q, r2 = tid / (C * Q);

    if (rank < natasks) PP::stage(p, rawsm, rank >> p.lgTPG, rank & TPGm);
    for (int a = rank; a < natasks; a += NA) {
        const int g = a >> p.lgTPG, tile = a & TPGm;
        const int n2_0 = tile * C;
        const int mg = g << p.lgGS;
        const int nsp = (p.nspec - mg < GS) ? p.nspec - mg : GS;
        float4* const zg = p.Z + ((size_t)((unsigned)g % (unsigned)p.RING) << p.lgGS) * N + n2_0 + c2;
        float2 tw[16];
        if (!DUMP) {
#pragma unroll
            for (int qb = 0; qb < 16; qb++) tw[qb] = __ldg(p.twT + (size_t)(qa * 16 + qb) * N2 + n2_0 + c2);
        }
        asm volatile("cp.async.wait_all;" ::: "memory");
        gsync<BAR, NT>();   // the staged tile is complete; the previous task's second stage has read ysm
        // ---------------- FIR phase (T = 1: unpack only)
#pragma unroll
        for (int i = 0; i < BPT; i++) {
            const int beta = tid + NT * i;
            if (T > 1) {
                const int nbr = (beta / C) * N2 + n2_0 + (beta % C);
                float hc[T];
#pragma unroll
                for (int t = 0; t < T; t++) hc[t] = __ldg(p.h + (size_t)t * N + nbr);
                cpx x[T];
#pragma unroll
                for (int t = 0; t < T - 1; t++) x[t] = unpack_cpx<2>(rawsm[t * BR + beta]);
#pragma unroll
                for (int r = 0; r < R; r++) {
                    x[(r + T - 1) % T] = unpack_cpx<2>(rawsm[(r + T - 1) * BR + beta]);
                    u64 re = 0ull, im = 0ull;
#pragma unroll
                    for (int t = 0; t < T; t++) {
                        re = fma2(x[(r + t) % T].re, bc(hc[t]), re);
                        im = fma2(x[(r + t) % T].im, bc(hc[t]), im);
                    }
                    ysm[r * BR + beta] = cpx_to_f4({re, im});
                }
            } else {
#pragma unroll
                for (int r = 0; r < R; r++) ysm[r * BR + beta] = cpx_to_f4(unpack_cpx<2>(rawsm[r * BR + beta]));
            }
        }
        if (!DUMP && tid == lead) wait_room(g);
        gsync<BAR, NT>();   // ysm complete, the raw tile is free again
        if (a + NA < natasks) PP::stage(p, rawsm, (a + NA) >> p.lgTPG, (a + NA) & TPGm);
        if (DUMP) {   // test hook: what the column transform is about to consume, in the caller's layout
            if (r2 < nsp) {
                float4* dp = (float4*)p.dump + (size_t)(mg + r2) * N + n2_0 + c2;
#pragma unroll
                for (int b = 0; b < 16; b++) {
                    const float4 z = ysm[(r2 * N1 + qa * 16 + b) * C + c2];
                    dp[(size_t)(qa * 16 + b) * N2] = make_float4(z.x, z.z, z.y, z.w);
                }
            }
        } else {
            // ---------------- first stage: radix Q over n1 = ja + 16 i, twiddle W_N1^{ja q}, in place
#pragma unroll
            for (int u = 0; u < 16 / Q; u++) {
                const int id = tid + NT * u;
                const int c = id % C, ja = (id / C) % 16, r = id / (16 * C);
                float4* y0 = ysm + (r * N1 + ja) * C + c;
                cpx v[Q];
#pragma unroll
                for (int i = 0; i < Q; i++) v[i] = f4_to_cpx(y0[i * 16 * C]);
                dft<Q>(v);
                y0[0] = cpx_to_f4(v[0]);
#pragma unroll
                for (int q = 1; q < Q; q++) {
                    const float2 w = __ldg(p.tw1 + (q - 1) * 16 + ja);
                    y0[q * 16 * C] = cpx_to_f4(cmul(v[q], w.x, w.y));
                }
            }
            gsync<BAR, NT>();
            // ---------------- second stage: radix 16 over block qa, W_N^{n2 k1}, rows p1 = 16 qa + qb of the Z ring
            if (r2 < nsp) {
                cpx v[16];
#pragma unroll
                for (int b = 0; b < 16; b++) v[b] = f4_to_cpx(ysm[(r2 * N1 + qa * 16 + b) * C + c2]);
                dft<16>(v);
                float4* zp = zg + (size_t)r2 * N + (size_t)(qa * 16) * N2;
#pragma unroll
                for (int qb = 0; qb < 16; qb++) zp[(size_t)qb * N2] = cpx_to_f4(cmul(v[qb], tw[qb].x, tw[qb].y));
            }
        }
        gsync<BAR, NT>();   // every Z store of the task has been issued by its thread; ysm may be overwritten
        if (!DUMP && tid == lead) signal(g, a + NA);
    }
}

// ---------------------------------------------------------------- A tasks in direct-FFT mode with the 16-point column DFT
// on the tensor cores (north_star: "Tensor cores may be used only for DFT factor stages that
// really are dense contractions, and only if the stated tolerance still holds").
// The int8 samples are exact in fp16; the real-ified DFT matrix (cos / sin of multiples of pi/8) is split into
// fp16 terms hi + mid (22 bits, the accuracy of an fp32 twiddle) that accumulate into the same fp32 tile:
//   D[128 x 64] = A[128 x 64] * B'[64 x 64]^T      per phase of 8 spectra x 16 columns, tcgen05.mma kind::f16, M = 128
//   row  = (spectrum fr, column fc) pair = thread id = TMEM lane
//   k    = pol*32 + 2*n1 + c            (c = 0 re, 1 im)       fp16 samples, K-major, no swizzle
//   col  = 4*k1 + {Xre, Yre, Xim, Yim}  -> tcgen05.ld hands every thread its 16 outputs as the packed pairs the
//                                          twiddle multiply and the Z store want
// B' is block diagonal in pol (half of its entries are zero: the tensor pipe is otherwise idle).  Shared memory:
// two A tiles of 16 KB (k-core major: [k/8][row/8][row%8][16 B], LBO = 2048, SBO = 128) and NSPLIT copies of B'
// (8 KB each: [k/8][col/8][col%8][16 B], LBO = 1024, SBO = 128); D is double-buffered in the 128 TMEM columns the
// producer CTAs allocate anyway.  The MMA of phase p+1 runs while the CTA twiddles and stores phase p.
constexpr int kTcSplit = 2;                         // fp16 terms of the DFT matrix
constexpr int kTcBBytes = kTcSplit * 64 * 64 * 2;   // bytes of B' in global / shared memory
constexpr size_t kTcSmem = 2 * 16384 + kTcBBytes + 64;

__device__ __forceinline__ uint64_t umma_desc(uint32_t saddr, uint32_t lbo, uint32_t sbo) {
    // K-major, no swizzle (cute::UMMA::SmemDescriptor: start >> 4 at [0,14), LBO >> 4 at [16,30), SBO >> 4 at [32,46),
    // version 1 at [46,48), layout type 0 at [61,64))
    return (uint64_t)((saddr & 0x3FFFFu) >> 4) | ((uint64_t)(lbo >> 4) << 16) | ((uint64_t)(sbo >> 4) << 32) | (1ull << 46);
}
__device__ __forceinline__ void umma_f16(uint32_t tmem_d, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t accumulate) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "setp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}"
        ::"r"(tmem_d), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate) : "memory");
}
__device__ __forceinline__ void umma_commit(uint64_t* bar) {
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
}

template <int NT, int N2, class WaitRoom, class Signal>
__device__ __forceinline__ void fused_producer_fft_tc(const FusedParams& p, float4* smem, uint32_t tmem_base, int rank, int NA,
                                                      int natasks, WaitRoom wait_room, Signal signal) {
    static_assert(NT == 128, "one MMA row per thread");
    constexpr int C = 16, R = NT / C, N = 16 * N2;
    uint8_t* const abuf = (uint8_t*)smem;                       // 2 x 16 KB
    uint8_t* const bsm = abuf + 2 * 16384;                      // kTcSplit x 8 KB
    uint64_t* const bar = (uint64_t*)(bsm + kTcBBytes);         // [2] MMA-complete barriers
    const int tid = threadIdx.x;
    const int GS = 1 << p.lgGS;
    const int TPGm = (1 << p.lgTPG) - 1;
    const int fr = tid / C, fc = tid % C;
    // instruction descriptor (cute::UMMA::InstrDescriptor): D = F32 at [4,6), A = B = F16 (0), K-major both, N >> 3 at [17,23), M >> 4 at [24,29)
    constexpr uint32_t idesc = (1u << 4) | ((64u >> 3) << 17) | ((128u >> 4) << 24);
    // TMEM address of my lane (lanes 32*(warp%4) .. +31 belong to this warp), column 0 of the CTA's allocation
    const uint32_t tlane = tmem_base + ((uint32_t)((tid >> 5) * 32) << 16);

    for (int i = tid; i < kTcBBytes / 16; i += NT) ((uint4*)bsm)[i] = __ldg((const uint4*)p.tcB + i);
    if (tid == 0) { mbar_init(&bar[0], 1); mbar_init(&bar[1], 1); }
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    __syncthreads();

    // the phases of my tasks, flattened: phase q of task a covers spectra mg + q*R .. of group g
    const int ppt = GS / R;                               // phases per task
    int nph = 0;
    for (int a = rank; a < natasks; a += NA) nph += ppt;
    auto phase_of = [&](int ph, int& a, int& j0) { a = rank + (ph / ppt) * NA; j0 = (ph % ppt) * R; };

    // convert + stage phase ph into A[ph & 1], then (thread 0) issue its MMAs into D[ph & 1]
    auto produce = [&](int ph) {
        int a, j0;
        phase_of(ph, a, j0);
        const int g = a >> p.lgTPG, tile = a & TPGm;
        const int mg = g << p.lgGS;
        const int nsp = (p.nspec - mg < GS) ? p.nspec - mg : GS;
        const int n2 = tile * C + fc;
        uint8_t* const arow = abuf + (ph & 1) * 16384 + (tid >> 3) * 128 + (tid & 7) * 16;
        uint32_t raw[16];
        const bool live = j0 + fr < nsp;
        const uint32_t* base = (const uint32_t*)p.view.in + (size_t)(mg + (live ? j0 + fr : 0)) * N + n2;
#pragma unroll
        for (int n1 = 0; n1 < 16; n1++) raw[n1] = live ? __ldg(base + n1 * N2) : 0u;
#pragma unroll
        for (int g4 = 0; g4 < 4; g4++) {
            uint32_t hx[4], hy[4];
#pragma unroll
            for (int i = 0; i < 4; i++) {
                // byte b (two's complement) -> fp16 bits 0x6400 | (b ^ 0x80) = 1024 + (b + 128); minus 1152: exact
                const uint32_t u = raw[4 * g4 + i] ^ 0x80808080u;
                const uint32_t px = __byte_perm(u, 0x64646464u, 0x4140);   // (Xre, Xim) as half2 bits
                const uint32_t py = __byte_perm(u, 0x64646464u, 0x4342);   // (Yre, Yim)
                asm("sub.rn.f16x2 %0, %1, %2;" : "=r"(hx[i]) : "r"(px), "r"(0x64806480u));   // 0x6480 = 1152.0
                asm("sub.rn.f16x2 %0, %1, %2;" : "=r"(hy[i]) : "r"(py), "r"(0x64806480u));
            }
            *(uint4*)(arow + g4 * 2048) = make_uint4(hx[0], hx[1], hx[2], hx[3]);          // k-cores 0..3: pol X
            *(uint4*)(arow + (4 + g4) * 2048) = make_uint4(hy[0], hy[1], hy[2], hy[3]);    // k-cores 4..7: pol Y
        }
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // my generic-proxy stores -> the tensor core's reads
        asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
        __syncthreads();
        if (tid == 0) {
            asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
            const uint32_t d = tmem_base + (uint32_t)((ph & 1) * 64);
            const uint32_t a0 = smem_u32(abuf + (ph & 1) * 16384);
#pragma unroll
            for (int sp = 0; sp < kTcSplit; sp++)
#pragma unroll
                for (int ks = 0; ks < 4; ks++)   // K = 64 in steps of 16 (two k-cores)
                    umma_f16(d, umma_desc(a0 + ks * 2 * 2048, 2048, 128), umma_desc(smem_u32(bsm) + sp * 8192 + ks * 2 * 1024, 1024, 128),
                             idesc, (sp | ks) ? 1u : 0u);
            umma_commit(&bar[ph & 1]);
        }
    };

    if (nph > 0) produce(0);
    float2 tw[16];
    for (int ph = 0; ph < nph; ph++) {
        int a, j0;
        phase_of(ph, a, j0);
        const int g = a >> p.lgTPG, tile = a & TPGm;
        const int mg = g << p.lgGS;
        const int nsp = (p.nspec - mg < GS) ? p.nspec - mg : GS;
        const int n2 = tile * C + fc;
        if (j0 == 0) {
#pragma unroll
            for (int k = 1; k < 16; k++) tw[k] = __ldg(p.twN + (size_t)n2 * k);
        }
        if (ph + 1 < nph) produce(ph + 1);   // staging + MMA of the next phase overlap this phase's epilogue
        if (j0 == 0) {   // first Z stores of a task: its ring slot must be free (the poll was issued a task ago)
            if (tid == 0) wait_room(g);
            __syncthreads();
        }
        // ---------------- epilogue of phase ph: D -> registers -> W_N twiddle -> Z ring
        mbar_wait(&bar[ph & 1], (ph >> 1) & 1);
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        float d0[32], d1[32];
        tmem_ld32(tlane + (uint32_t)((ph & 1) * 64), d0);
        tmem_ld32(tlane + (uint32_t)((ph & 1) * 64 + 32), d1);
        tmem_wait_ld();
        asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
        if (j0 + fr < nsp) {
            float4* zp = p.Z + ((size_t)((unsigned)g % (unsigned)p.RING) << p.lgGS) * N + (size_t)(j0 + fr) * N + n2;
            zp[0] = make_float4(d0[0], d0[1], d0[2], d0[3]);
#pragma unroll
            for (int k = 1; k < 16; k++) {
                const float* d = (k < 8) ? d0 + 4 * k : d1 + 4 * (k - 8);
                const cpx v = cmul({pk(d[0], d[1]), pk(d[2], d[3])}, tw[k].x, tw[k].y);
                zp[k * N2] = cpx_to_f4(v);
            }
        }
        if (j0 + R >= GS || ph + 1 == nph) {   // last phase of a task: publish it
            __syncthreads();   // every Z store of the task has been issued by its thread
            if (tid == 0) signal(g, a + NA);
        }
    }
}

// ---------------------------------------------------------------- the kernel
//   TC (direct-FFT mode, N1 = 16, NT = 128): the producers' 16-point column DFT runs on the tensor cores
template <class PL, int NT, int MODE_PFB, int PER_SM, bool DUMP = false, int N1 = 16, bool TC = false>
__global__ void __launch_bounds__(NT, PER_SM)
k_fused(const FusedParams p) {
    constexpr int L = PL::L, RA = PL::RA, RB = PL::RB, RC = PL::RC, NST = PL::NST;
    constexpr int LA = PL::LA, LB = PL::LB, NTS = PL::NTS;
    constexpr int G = NT / NTS;                     // rows per B job
    constexpr int RGN = (G >= N1) ? 1 : N1 / G;     // row groups per spectrum (a spectrum has N1 rows)
    constexpr int SPJ = (G >= N1) ? G / N1 : 1;     // spectra per B job
    constexpr int NSETS = NT / 128;                 // tensor memory: one block of 128 columns per set of four warps (64 accumulator + 64 twiddle columns)
    static_assert(NST >= 2 && PL::RLAST == 16 && G * L * 16 == NT * 256, "row plan");
    extern __shared__ float4 smem[];                // G*L float4: B exchange buffer / A FIR hand-off (+ the staged raw tile)
    __shared__ int s_role[2];
    __shared__ uint32_t s_tmem[NSETS];

    const int tid = threadIdx.x;
    const int GS = 1 << p.lgGS;
    const int ngroups = (p.nspec + GS - 1) >> p.lgGS;
    const unsigned TPG = 1u << p.lgTPG;
    const unsigned a_full = TPG;                    // a_done of a complete group
    const unsigned rows_full = (unsigned)GS * (unsigned)N1;

    if (DUMP) {
        // Test hook: every CTA runs the producer's front end on the tasks blockIdx.x, blockIdx.x + gridDim.x, ...
        // and writes what it would hand to the column FFT; no roles, no tensor memory, no counters, and no CTA
        // waits for another (this instantiation needs fewer registers, so more CTAs than PER_SM may share an SM).
        const int natasks = ngroups << p.lgTPG;
        auto no_wait = [](int) {};
        if constexpr (N1 > 16) {
            fused_producer_big<NT, L, N1, MODE_PFB ? 8 : 1, true>(p, smem, (int)blockIdx.x, (int)gridDim.x, natasks, no_wait,
                                                                  [](int, int) {}, 0);
        } else if (MODE_PFB) {
            fused_producer_pfb<NT, L, true>(p, smem, (int)blockIdx.x, (int)gridDim.x, natasks, no_wait, [](int, int) {});
        } else {
            for (int a = blockIdx.x; a < natasks; a += gridDim.x)
                fused_task_A_fft<NT, L, true>(p, a >> p.lgTPG, a & (int)(TPG - 1), no_wait);
        }
        return;
    }
    // Every CTA allocates its TMEM columns first, producers included: a CTA of a kernel that contains
    // tcgen05.alloc holds the SM's allocation permit until it relinquishes it, and (measured) no
    // further CTA of the grid is started on that SM before then.
    tmem_alloc_sets<NSETS>(s_tmem);
    const uint32_t tmem_base = *(volatile uint32_t*)&s_tmem[0];                    // (the tensor-core producer's tile: NT = 128)
    const uint32_t tmem_mine = *(volatile uint32_t*)&s_tmem[threadIdx.x >> 7];     // my set's block

    // role and rank: the first na_per_sm CTAs to arrive on an SM produce, the others consume
    if (tid == 0) {
        unsigned smid;
        asm volatile("mov.u32 %0, %%smid;" : "=r"(smid));
        const unsigned li = atomicAdd(p.role + 4 + smid, 1u);
        const int is_a = li < (unsigned)p.na_per_sm;
        s_role[0] = is_a;
        s_role[1] = (int)atomicAdd(p.role + (is_a ? 0 : 1), 1u);
        atomicAdd(p.role + 2, 1u);   // arrivals
        // The history this launch reads was written by the previous launch's CTAs (the carry below), and the two
        // launches overlap: acquire it through the carry counter instead of relying on stream order.  (The
        // counter is complete long before any CTA of this launch starts: the previous launch triggers its
        // dependents only after every one of its CTAs has signalled.)
        if (p.carry_wait_on && is_a) {
            wait_counter_wrap(p.carry_cnt, p.carry_wait, p.err);
            fence_acquire_gpu();
        }
    }
    // the history of the next call (the (T-1)*N samples carried across calls), one chunk per thread;
    // it goes to a buffer that neither this launch nor the previous one reads (three buffers rotate)
    for (int i = blockIdx.x * NT + tid; i < p.carry_chunks; i += gridDim.x * NT) p.carry_dst[i] = __ldg(p.carry_src + i);
    __syncthreads();
    if (p.carry_chunks && tid == 0) red_release_u32(p.carry_cnt, 1u);   // (cumulative over the CTA's stores)
    // Programmatic dependent launch: the next spec_process call's launch (same stream, launched with
    // programmatic stream serialisation) may start filling SM slots as soon as EVERY CTA of this grid is
    // resident and has carried its share of the history; its CTAs then land in the slots this grid's CTAs
    // free one by one (producers leave first, and the first arrivals on an SM produce), so the next call's
    // pipeline fills while this call's consumers drain.  The two launches share the accumulators (atomic
    // adds) and the history buffer this launch has just written (acquired by the next launch through
    // carry_cnt); Z rings and counters alternate between launches, the history rotates through three
    // buffers (the next launch writes the one neither of the two reads), and a third launch cannot start
    // before this one is gone (its predecessor is not fully resident until then: the grid is exactly what
    // the SMs hold).
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    // No CTA may leave before every CTA of the grid has arrived: an early exit would free a slot on its
    // SM, a late CTA would land there as a fifth arrival and the per-SM role split would be off.
    auto finish = [&]() {
        __syncthreads();
        // (the previous launch, if this one overlapped its tail, has completed long before any CTA gets here;
        // waiting for it formally keeps completion in stream order)
        asm volatile("griddepcontrol.wait;" ::: "memory");
        if (tid == 0) {
            wait_counter(p.role + 2, gridDim.x, p.err);
            __threadfence();
            s_role[0] = (atomicAdd(p.role + 3, 1u) == gridDim.x - 1);   // am I the last one out?
        }
        __syncthreads();
        if (s_role[0]) {
            __threadfence();
            for (int i = tid; i < ngroups; i += NT) { p.a_done[i] = 0u; p.b_done[i] = 0u; }
            for (int i = tid; i < kFusedRoleWords; i += NT) p.role[i] = 0u;
        }
        tmem_free_sets<NSETS>(s_tmem);
    };
    const bool is_a = s_role[0] != 0;
    const int rank = s_role[1];
    const int lead = 0;   // the CTA's polling / signalling thread (moving it to warp rank % 4 measured no gain)
    const int per_sm = PER_SM;
    const int nsm = (int)gridDim.x / per_sm;
    // thread 0's polls are issued one task ahead into a register (pf_val: the counter of group pf_g)
    unsigned pf_val = 0u;
    int pf_g = -1;

    if (is_a) {
        // ================= producer: A tasks rank, rank + NA, ...
        const int NA = nsm * p.na_per_sm;
        const int natasks = ngroups << p.lgTPG;
        int room_g = -1;   // thread 0: newest group whose ring slot is known to be free
        auto wait_room = [&](int g) {
            const int gfree = g - p.RING;     // the group whose ring slot this task overwrites
            if (gfree < 0 || gfree <= room_g) return;
            if (!(pf_g == gfree && pf_val >= rows_full)) wait_counter(p.b_done + gfree, rows_full, p.err);
            fence_acquire_task();   // the consumers' reads of the slot happen before my CTA's stores (after the barrier)
            room_g = gfree;
        };
        auto prefetch_room = [&](int a) {    // thread 0, for my task a (if any)
            if (a < natasks && (a >> p.lgTPG) >= p.RING && (a >> p.lgTPG) - p.RING > room_g) {
                pf_g = (a >> p.lgTPG) - p.RING;
                pf_val = ld_relaxed_u32(p.b_done + pf_g);
            }
        };
        if constexpr (N1 > 16) {
            if (tid == lead) prefetch_room(rank);
            fused_producer_big<NT, L, N1, MODE_PFB ? 8 : 1, false>(p, smem, rank, NA, natasks, wait_room, [&](int g, int a_next) {
                red_release_u32(p.a_done + g, 1u);   // all Z stores of the CTA are ordered before it
                prefetch_room(a_next);
            }, lead);
        } else if (MODE_PFB) {
            if (tid == lead) prefetch_room(rank);
            fused_producer_pfb<NT, L, false>(p, smem, rank, NA, natasks, wait_room, [&](int g, int a_next) {
                red_release_u32(p.a_done + g, 1u);   // all Z stores of the CTA are ordered before it
                prefetch_room(a_next);
            }, lead);
        } else if constexpr (TC) {
            if (tid == 0) prefetch_room(rank);
            fused_producer_fft_tc<NT, L>(p, smem, tmem_base, rank, NA, natasks, wait_room, [&](int g, int a_next) {
                red_release_u32(p.a_done + g, 1u);
                prefetch_room(a_next);
            });
        } else {
            for (int a = rank; a < natasks; a += NA) {
                const int g = a >> p.lgTPG;
                if (tid == lead) prefetch_room(a);
                fused_task_A_fft<NT, L, false>(p, g, a & (int)(TPG - 1), wait_room, lead);   // ends with a __syncthreads
                if (tid == lead) red_release_u32(p.a_done + g, 1u);
            }
        }
        finish();
        return;
    }

    // ================= consumer: row group rg of the jobs y, y+ny, y+2ny, ...  (job j = spectra j*SPJ ..)
    const int NB = nsm * (per_sm - p.na_per_sm);
    const int slot = tid / NTS, t = tid % NTS;
    const int RS = p.RING << p.lgGS;                // spectra in the Z ring
    const int rg = rank % RGN;
    const int y = rank / RGN;
    const int ny = NB / RGN;
    const int njobs_all = (p.nspec + SPJ - 1) / SPJ;
    const int nbj = (y < ny && y < njobs_all) ? (njobs_all - y + ny - 1) / ny : 0;  // my B jobs
    const int row = (G >= N1) ? (slot % N1) : (rg * G + slot);
    const int sub = (G >= N1) ? (slot / N1) : 0;    // which spectrum of the job this slot works on
    const int mstride = ny * SPJ;
    const int zstride = mstride % RS;
    int m = y * SPJ + sub;                          // spectrum of my next job for this slot
    int zpos = m % RS;                              // its ring position
    auto addr = [&](int q) -> int { return slot * L + (q ^ ((q / 16) & 7)); };
    // The same swizzle written out for the three-stage plans (LA = 256, LB = RB = RC = 16), so that the 16
    // addresses of a stage are one base plus compile-time offsets plus one of the 8 values (t & 7) ^ k,
    // instead of 16 independent registers per stage (which ptxas hoists out of the job loop and spills):
    //   stage a: q = ja + qq*LA, LA % 128 == 0  =>  addr(q) = addr(ja) + qq*LA
    //   stage b: q = (t/16)*LA + t%16 + 16 r     =>  (q/16) & 7 = r & 7, the XOR touches t%16 only
    //   stage c: q = 16 t + r                    =>  (q/16) & 7 = t & 7, the XOR touches r only
    const int c7 = t & 7;
    const int bbase = slot * L + (t >> 4) * LA + (t & 8);
    const int cbase = slot * L + 16 * t;
    auto addr_b = [&](int r) -> int { return bbase + 16 * r + (c7 ^ (r & 7)); };
    auto addr_c = [&](int r) -> int { return cbase + (r & 8) + (c7 ^ (r & 7)); };
    constexpr bool kExplicit = (NST == 3) && (LA % 128 == 0) && (LB == 16) && (RB == 16) && (RC == 16);
    auto group_of_job = [&](int j) -> int {
        int s1 = (y + j * ny) * SPJ + SPJ - 1;
        if (s1 > p.nspec - 1) s1 = p.nspec - 1;
        return s1 >> p.lgGS;
    };

    SinkStokesTmem sink{p.ring, p.acc_stride, p.nring, L, 1};
    SinkStokesTmem::State st;
    sink.init_set(st, tmem_mine);
    sink.begin(st);
    // The stage twiddles a thread needs are the same for every job (they depend on its index only):
    // they are parked in tensor memory next to the accumulators (columns 64.. of the thread's lane) and
    // fetched with one tcgen05.ld per stage, instead of 29 global loads per job that mostly missed the
    // small L1 left beside the shared-memory carve-out (measured: 14 of 40 B/sample of L2->SM traffic).
    constexpr int TWA = (16 / RA) * (RA - 1);                       // float2 per thread, stage a
    constexpr int TWB = (NST == 3) ? (16 / RB) * (RB - 1) : 0;      // stage b
    static_assert(TWA <= 16 && TWB <= 16, "32 words per stage");
    const uint32_t ttw = st.taddr + 64;
    {
        float w[32];
#pragma unroll
        for (int i = 0; i < 32; i++) w[i] = 0.f;
#pragma unroll
        for (int u = 0; u < 16 / RA; u++)
#pragma unroll
            for (int q = 1; q < RA; q++) {
                const float2 x = __ldg(p.twL + (q - 1) * LA + t + NTS * u);
                w[2 * (u * (RA - 1) + q - 1)] = x.x;
                w[2 * (u * (RA - 1) + q - 1) + 1] = x.y;
            }
        tmem_st32(ttw, w);
        if (NST == 3) {
            float w2[32];
#pragma unroll
            for (int i = 0; i < 32; i++) w2[i] = 0.f;
#pragma unroll
            for (int u = 0; u < 16 / RB; u++)
#pragma unroll
                for (int q = 1; q < RB; q++) {
                    const float2 x = __ldg(p.twL + (RA - 1) * LA + (q - 1) * LB + (t + NTS * u) % LB);
                    w2[2 * (u * (RB - 1) + q - 1)] = x.x;
                    w2[2 * (u * (RB - 1) + q - 1) + 1] = x.y;
                }
            tmem_st32(ttw + 32, w2);
        }
        tmem_wait_st();
    }
    long long wcur = -1;       // accumulation window the TMEM sums belong to (-1: none yet)
    long long nextb = 0;       // first spectrum (of this launch) that no longer belongs to window wcur
    int ready_g = -1;          // thread 0: newest group known to be complete

    // CTA-wide synchronisation of a job: ONE barrier (after stage a's exchange stores).  The write-after-
    // read hazard on the exchange buffer (stage a of job i+1 overwrites what the last stage of job i
    // reads) is covered by a split-phase mbarrier instead of a second barrier: a thread arrives once its
    // last butterfly has consumed its loads and only waits just before its next exchange stores, with
    // the TMEM update, the window check, the row loads and the first butterflies in between.
    __shared__ uint64_t s_war;
    if (tid == 0) mbar_init(&s_war, NT);
    auto wait_ready = [&](int j) {       // thread 0: returns once the group of my job j is complete
        const int g = group_of_job(j);
        if (g == ready_g) return;
        if (!(pf_g == g && pf_val >= a_full)) wait_counter(p.a_done + g, a_full, p.err);
        fence_acquire_task();   // (published to the other threads by the CTA barrier that follows)
        ready_g = g;
    };
    auto prefetch_ready = [&](int j) {   // thread 0
        if (j < nbj) {
            const int g = group_of_job(j);
            if (g != ready_g) { pf_g = g; pf_val = ld_relaxed_u32(p.a_done + g); }
        }
    };
    if (tid == lead && nbj > 0) { prefetch_ready(0); wait_ready(0); prefetch_ready(1); }
    __syncthreads();
    for (int bi = 0; bi < nbj; bi++) {
        // ---------------- B job bi: spectrum m (ring position zpos), row `row`
        const bool active = m < p.nspec;
        if (active && m >= nextb) {   // new accumulation window (warp-uniform: a warp never straddles spectra)
            if (wcur >= 0) { sink.flush(st, row, t, wcur); sink.begin(st); }
            wcur = (p.c0 + m) / p.M;
            nextb = (wcur + 1) * p.M - p.c0;
        }
        const float4* zrow = p.Z + (size_t)zpos * (N1 * L) + row * L;
        // stage a: rows of Z straight from L2 (ld.global.cg: the ring is rewritten by other SMs)
        if (active) {
            float twa[32];
            tmem_ld32(ttw, twa);
            cpx v[16 / RA][RA];
#pragma unroll
            for (int u = 0; u < 16 / RA; u++)
#pragma unroll
                for (int r = 0; r < RA; r++) v[u][r] = f4_to_cpx(__ldcg(zrow + t + NTS * u + r * LA));
            tmem_wait_ld();
            if (bi > 0) mbar_wait(&s_war, (bi - 1) & 1);   // everybody is done reading the previous job
#pragma unroll
            for (int u = 0; u < 16 / RA; u++) {
                const int ja = t + NTS * u;
                const int aja = addr(ja);
                dft<RA>(v[u]);
                smem[aja] = cpx_to_f4(v[u][0]);
#pragma unroll
                for (int q = 1; q < RA; q++)
                    smem[kExplicit ? aja + q * LA : addr(ja + q * LA)] =
                        cpx_to_f4(cmul(v[u][q], twa[2 * (u * (RA - 1) + q - 1)], twa[2 * (u * (RA - 1) + q - 1) + 1]));
            }
        } else if (bi > 0) {
            mbar_wait(&s_war, (bi - 1) & 1);
        }
        // the next job's group must be complete before anybody loads its rows: checked here (the poll
        // was prefetched a job ago), published by the barrier
        if (tid == lead && bi + 1 < nbj) { wait_ready(bi + 1); prefetch_ready(bi + 2); }
        __syncthreads();
        // The rows just consumed are dead (their ring slot will be rewritten in full): drop their dirty L2
        // lines instead of letting them be written back to HBM -- the ring is meant to live in L2 only.
        if (active) {
#pragma unroll
            for (int i = 0; i < (L * 16) / (NTS * 128); i++)
                asm volatile("discard.global.L2 [%0], 128;" ::"l"(zrow + (t + NTS * i) * 8) : "memory");
        }
        if (tid == lead) {   // my rows of this job are consumed: the producers may reuse the ring slot
            const int s0 = (y + bi * ny) * SPJ;
            int s1 = s0 + SPJ;
            if (s1 > p.nspec) s1 = p.nspec;
            // (a job of several spectra never straddles groups: SPJ divides GS)
            red_release_u32(p.b_done + (s0 >> p.lgGS), (G >= N1) ? (unsigned)(N1 * (s1 - s0)) : (unsigned)G);
        }
        if (active) {
            float twb[32];
            if (NST == 3) tmem_ld32(ttw + 32, twb);
#pragma unroll
            for (int u = 0; u < 16 / RB; u++) {
                const int i = t + NTS * u;
                const int qa = i / LB, jb = i % LB;
                const int base = qa * LA + jb;
                cpx v[RB];
#pragma unroll
                for (int r = 0; r < RB; r++) v[r] = f4_to_cpx(smem[kExplicit ? addr_b(r) : addr(base + r * LB)]);
                if (NST == 2) mbar_arrive(&s_war);   // (release: my reads of the exchange buffer are done)
                dft<RB>(v);
                if (NST == 2) {
                    sink.put16(st, m, 0, i, i, RA, v);
                } else {
                    if (u == 0) tmem_wait_ld();
                    smem[kExplicit ? addr_b(0) : addr(base)] = cpx_to_f4(v[0]);
#pragma unroll
                    for (int q = 1; q < RB; q++)
                        smem[kExplicit ? addr_b(q) : addr(base + q * LB)] = cpx_to_f4(cmul(v[q], twb[2 * (u * (RB - 1) + q - 1)],
                                                                  twb[2 * (u * (RB - 1) + q - 1) + 1]));
                }
            }
        }
        if (NST == 3) {
            // stage b -> c only exchanges data inside groups of LB = 16 adjacent threads (one block of
            // LA points), so a warp-level barrier is enough
            static_assert(NST != 3 || (LB == 16 && RC == 16), "stage c reads what its own half-warp wrote");
            __syncwarp();
            if (active) {
                float a0[32];
                sink.preload(st, a0);   // first half of my accumulators, in flight during the butterfly
                cpx v[RC];
#pragma unroll
                for (int r = 0; r < RC; r++) v[r] = f4_to_cpx(smem[kExplicit ? addr_c(r) : addr(t * RC + r)]);
                mbar_arrive(&s_war);   // (release: my reads of the exchange buffer are done)
                dft<RC>(v);
                sink.put16_preloaded(st, a0, v);
            }
        }
        if (!active) mbar_arrive(&s_war);
        m += mstride;
        zpos += zstride;
        if (zpos >= RS) zpos -= RS;
    }
    if (wcur >= 0) sink.flush(st, row, t, wcur);
    finish();
}

}  // namespace spk
