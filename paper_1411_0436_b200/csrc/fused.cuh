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
// (cumulative over the CTA's stores); the reader's poll is a relaxed (strong) load, made an acquire by this
// fence, and the CTA barrier that follows extends the ordering to the other threads of the reader.
#ifndef SPK_ACQ_FENCE
#define SPK_ACQ_FENCE 1
#endif
#ifndef SPK_LEADER_ROT
#define SPK_LEADER_ROT 0   // 1: the polling / signalling thread of a CTA sits in warp (rank mod warps) instead of warp 0
#endif
__device__ __forceinline__ void fence_acquire_gpu() {
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
template <int NT, int N2, bool DUMP, class WaitRoom, class Signal>
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
            __syncthreads();   // the staged tile is complete; the previous phase's column FFTs have read ysm
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
            __syncthreads();   // ysm complete, the raw tile is free again
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
        __syncthreads();   // every Z store of the task has been issued by its thread
        if (!DUMP && tid == lead) signal(g, a + NA);
    }
}

// One A task in direct-FFT mode: no pre-filter, the 16 samples of a column go straight
// from global memory through the unpack into the butterfly.
template <int NT, int N2, bool DUMP, class WaitRoom>
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
    __syncthreads();
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
    __syncthreads();
}

// ---------------------------------------------------------------- the kernel
template <class PL, int NT, int MODE_PFB, int PER_SM, bool DUMP = false>
__global__ void __launch_bounds__(NT, PER_SM)
k_fused(const FusedParams p) {
    constexpr int L = PL::L, RA = PL::RA, RB = PL::RB, RC = PL::RC, NST = PL::NST;
    constexpr int LA = PL::LA, LB = PL::LB, NTS = PL::NTS;
    constexpr int G = NT / NTS;                     // rows per B job
    constexpr int RGN = (G >= 16) ? 1 : 16 / G;     // row groups per spectrum
    constexpr int SPJ = (G >= 16) ? G / 16 : 1;     // spectra per B job
    constexpr int TCOLS = (NT > 128) ? 256 : 128;   // per set of four warps: 64 accumulator + 64 twiddle columns
    static_assert(NST >= 2 && PL::RLAST == 16 && G * L * 16 == NT * 256, "row plan");
    extern __shared__ float4 smem[];                // G*L float4: B exchange buffer / A FIR hand-off (+ the staged raw tile)
    __shared__ int s_role[2];
    __shared__ uint32_t s_tmem;

    const int tid = threadIdx.x;
    const int GS = 1 << p.lgGS;
    const int ngroups = (p.nspec + GS - 1) >> p.lgGS;
    const unsigned TPG = 1u << p.lgTPG;
    const unsigned a_full = TPG;                    // a_done of a complete group
    const unsigned rows_full = (unsigned)GS * 16u;

    if (DUMP) {
        // Test hook: every CTA runs the producer's front end on the tasks blockIdx.x, blockIdx.x + gridDim.x, ...
        // and writes what it would hand to the column FFT; no roles, no tensor memory, no counters, and no CTA
        // waits for another (this instantiation needs fewer registers, so more CTAs than PER_SM may share an SM).
        const int natasks = ngroups << p.lgTPG;
        auto no_wait = [](int) {};
        if (MODE_PFB) {
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
    const uint32_t tmem_base = tmem_alloc_cta<TCOLS>(&s_tmem);

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
    const uint32_t tmem_base_ = tmem_base;
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
        tmem_free_cta<TCOLS>(tmem_base_);
    };
    const bool is_a = s_role[0] != 0;
    const int rank = s_role[1];
    const int lead = SPK_LEADER_ROT ? 32 * (rank % (NT / 32)) : 0;   // the CTA's polling / signalling thread
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
            fence_acquire_gpu();   // the consumers' reads of the slot happen before my CTA's stores (after the barrier)
            room_g = gfree;
        };
        auto prefetch_room = [&](int a) {    // thread 0, for my task a (if any)
            if (a < natasks && (a >> p.lgTPG) >= p.RING && (a >> p.lgTPG) - p.RING > room_g) {
                pf_g = (a >> p.lgTPG) - p.RING;
                pf_val = ld_relaxed_u32(p.b_done + pf_g);
            }
        };
        if (MODE_PFB) {
            if (tid == lead) prefetch_room(rank);
            fused_producer_pfb<NT, L, false>(p, smem, rank, NA, natasks, wait_room, [&](int g, int a_next) {
                red_release_u32(p.a_done + g, 1u);   // all Z stores of the CTA are ordered before it
                prefetch_room(a_next);
            }, lead);
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
    const int row = (G >= 16) ? (slot % 16) : (rg * G + slot);
    const int sub = (G >= 16) ? (slot / 16) : 0;    // which spectrum of the job this slot works on
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
    sink.init(st, tmem_base, 128);
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
        fence_acquire_gpu();   // (published to the other threads by the CTA barrier that follows)
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
        const float4* zrow = p.Z + (size_t)zpos * (16 * L) + row * L;
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
            red_release_u32(p.b_done + (s0 >> p.lgGS), (G >= 16) ? (unsigned)(16 * (s1 - s0)) : (unsigned)G);
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
