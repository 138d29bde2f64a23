// fused2.cuh — the persistent four-step kernel with BOTH roles in every CTA (N = 16 x N2, N2 = 512, 1024, 2048).
//
// Same algorithm, ring and counters as k_fused (fused.cuh); what changes is how the roles share an SM:
//   * a CTA is 256 threads: warps 0-3 are a PRODUCER group (A tasks, unchanged code, named barrier 1), warps 4-7 a
//     CONSUMER group (B jobs, named barrier 2); two such CTAs per SM give the same 2 + 2 split k_fused gets from
//     the order of arrival, but fixed by construction: no per-SM arrival counters, no "nobody leaves before
//     everybody has arrived";
//   * shared memory is no longer the same for both roles: the consumer group owns TWO row buffers of 32 KB, and
//     the rows of its NEXT job arrive in the idle one by cp.async.bulk (one elected thread, mbarrier completion)
//     while it computes the current job.  The row loads (ld.global.cg, an L2 round trip per job that every warp
//     of the group waited for, each for its own rows, before the group barrier) are gone from the warps;
//   * the landed rows are transformed IN PLACE: stage a reads them in natural order and writes the swizzled
//     exchange layout back into the same buffer (the permutation stays inside aligned groups of eight lanes, so a
//     __syncwarp between the loads and the stores is enough), stages b and c work in place as before.  The
//     buffer of job i-1 is free once every thread has passed job i's group barrier, which is when the elected
//     thread issues the copy for job i+1;
//   * a ring slot is released (b_done) as soon as its rows have landed in shared memory.
#pragma once
#include "fused.cuh"

namespace spk {

// NT = threads per role group: 128 (N2 <= 2048, two CTAs per SM) or 256 (N2 = 4096: N = 65536 and, with the
// N1 = 32 / 64 / 128 column plans of ProducerBig, N >= 131072; one CTA of 512 threads per SM)
template <class PL, int MODE_PFB, int N1>
struct Fused2Shape {
    static constexpr int NT = (PL::L == 4096) ? 256 : 128;
    static constexpr int G = NT / PL::NTS;                           // rows per B job
    static constexpr size_t P16 = MODE_PFB ? (size_t)NT * 16 * sizeof(float4) + (size_t)(NT / 16 + 7) * 1024 : 0;
    static constexpr size_t PBIG = ProducerBig<256, PL::L, (N1 > 16 ? N1 : 32), MODE_PFB ? 8 : 1>::SMEM;
    static constexpr size_t P_BYTES = (N1 > 16) ? PBIG : P16;
    static constexpr size_t ROW_BYTES = (size_t)G * PL::L * sizeof(float4);   // one job's rows: 32 or 64 KB
    static constexpr size_t SMEM = P_BYTES + 2 * ROW_BYTES;
    static constexpr bool kFits = SMEM + 2048 <= 227 * 1024 / (256 / NT);
};

template <class PL, int MODE_PFB, int N1 = 16>
__global__ void __launch_bounds__(2 * Fused2Shape<PL, MODE_PFB, N1>::NT, 256 / Fused2Shape<PL, MODE_PFB, N1>::NT)
k_fused2(const FusedParams p) {
    typedef Fused2Shape<PL, MODE_PFB, N1> SH;
    constexpr int NT = SH::NT;
    constexpr int NTC = 2 * NT;                     // threads per CTA
    constexpr int NSETS = NT / 128;                 // tensor memory: one block of 128 columns per set of four CONSUMER warps
    constexpr int L = PL::L, RA = PL::RA, RB = PL::RB, RC = PL::RC, NST = PL::NST;
    constexpr int LA = PL::LA, LB = PL::LB, NTS = PL::NTS;
    constexpr int G = SH::G;
    constexpr int RGN = N1 / G;                     // row groups per spectrum (a spectrum has N1 rows)
    static_assert(NST == 3 && LB == 16 && RB == 16 && RC == 16 && LA % 128 == 0 && G >= 1 && G < N1, "three-stage row plan");
    extern __shared__ float4 smem[];
    float4* const rowbuf = (float4*)((uint8_t*)smem + SH::P_BYTES);   // [2][G*L]
    __shared__ uint32_t s_tmem[NSETS];
    __shared__ uint64_t s_full[2];
    __shared__ int s_last;

    const int gtid = threadIdx.x;
    const bool is_a = gtid < NT;
    const int tid = gtid & (NT - 1);
    const int GS = 1 << p.lgGS;
    const int ngroups = (p.nspec + GS - 1) >> p.lgGS;
    const unsigned TPG = 1u << p.lgTPG;
    const unsigned a_full = TPG;
    const unsigned rows_full = (unsigned)GS * (unsigned)N1;

    // (blocks of 128 columns only: see tmem_alloc_sets in engine.cuh; the producer warps use none)
    tmem_alloc_sets<NSETS>(s_tmem);
    const uint32_t tmem_mine = *(volatile uint32_t*)&s_tmem[is_a ? 0 : (gtid - NT) >> 7];
    if (gtid == 0) {
        mbar_init(&s_full[0], 1);
        mbar_init(&s_full[1], 1);
        if (p.carry_wait_on) {   // the history the previous (overlapping) launch wrote: acquire it (fused.cuh)
            wait_counter_wrap(p.carry_cnt, p.carry_wait, p.err);
            fence_acquire_gpu();
        }
    }
    for (int i = blockIdx.x * NTC + gtid; i < p.carry_chunks; i += gridDim.x * NTC) p.carry_dst[i] = __ldg(p.carry_src + i);
    __syncthreads();
    if (p.carry_chunks && gtid == 0) red_release_u32(p.carry_cnt, 1u);
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");

    const int rank = blockIdx.x;          // of my group among the groups of its kind
    const int ngrp = gridDim.x;           // producer groups == consumer groups == CTAs
    unsigned pf_val = 0u;                 // the group leader's poll, issued one task ahead
    int pf_g = -1;

    if (is_a) {
        // ================= producer group: A tasks rank, rank + ngrp, ...
        const int natasks = ngroups << p.lgTPG;
        int room_g = -1;
        auto wait_room = [&](int g) {
            const int gfree = g - p.RING;
            if (gfree < 0 || gfree <= room_g) return;
            if (!(pf_g == gfree && pf_val >= rows_full)) wait_counter(p.b_done + gfree, rows_full, p.err);
            fence_acquire_task();
            room_g = gfree;
        };
        auto prefetch_room = [&](int a) {
            if (a < natasks && (a >> p.lgTPG) >= p.RING && (a >> p.lgTPG) - p.RING > room_g) {
                pf_g = (a >> p.lgTPG) - p.RING;
                pf_val = ld_relaxed_u32(p.b_done + pf_g);
            }
        };
        auto signal = [&](int g, int a_next) {
            red_release_u32(p.a_done + g, 1u);   // all Z stores of the group are ordered before it
            prefetch_room(a_next);
        };
        if constexpr (N1 > 16) {
            if (tid == 0) prefetch_room(rank);
            fused_producer_big<NT, L, N1, MODE_PFB ? 8 : 1, false, decltype(wait_room), decltype(signal), 1>(
                p, smem, rank, ngrp, natasks, wait_room, signal, 0);
        } else if (MODE_PFB) {
            if (tid == 0) prefetch_room(rank);
            fused_producer_pfb<NT, L, false, decltype(wait_room), decltype(signal), 1>(p, smem, rank, ngrp, natasks, wait_room, signal, 0);
        } else {
            for (int a = rank; a < natasks; a += ngrp) {
                const int g = a >> p.lgTPG;
                if (tid == 0) prefetch_room(a);
                fused_task_A_fft<NT, L, false, decltype(wait_room), 1>(p, g, a & (int)(TPG - 1), wait_room, 0);
                if (tid == 0) red_release_u32(p.a_done + g, 1u);
            }
        }
    } else {
        // ================= consumer group: row group rg of the spectra y, y + ny, ...
        const int slot = tid / NTS, t = tid % NTS;
        const int RS = p.RING << p.lgGS;                // spectra in the Z ring
        const int rg = rank % RGN, y = rank / RGN, ny = ngrp / RGN;
        const int nbj = (y < ny && y < p.nspec) ? (p.nspec - y + ny - 1) / ny : 0;   // my B jobs (one spectrum each)
        const int row = rg * G + slot;
        const int zstride = ny % RS;
        int m = y;                                      // spectrum of my next job
        int zpos = m % RS;                              // its ring position
        // swizzled exchange layout inside a row buffer (engine.cuh): address of natural position q of my slot
        const int c7 = t & 7;
        const int bbase = slot * L + (t >> 4) * LA + (t & 8);
        const int cbase = slot * L + 16 * t;
        auto addr_b = [&](int r) -> int { return bbase + 16 * r + (c7 ^ (r & 7)); };
        auto addr_c = [&](int r) -> int { return cbase + (r & 8) + (c7 ^ (r & 7)); };

        SinkStokesTmem sink{p.ring, p.acc_stride, p.nring, L, 1};
        SinkStokesTmem::State st;
        sink.init_set(st, tmem_mine);
        sink.begin(st);
        // the thread's stage twiddles, parked in tensor memory next to its accumulators (fused.cuh)
        constexpr int TWA = (16 / RA) * (RA - 1);
        constexpr int TWB = (16 / RB) * (RB - 1);
        static_assert(TWA <= 16 && TWB <= 16, "32 words per stage");
        const uint32_t ttw = st.taddr + 64;
        {
            float w[32], w2[32];
#pragma unroll
            for (int i = 0; i < 32; i++) { w[i] = 0.f; w2[i] = 0.f; }
#pragma unroll
            for (int u = 0; u < 16 / RA; u++)
#pragma unroll
                for (int q = 1; q < RA; q++) {
                    const float2 x = __ldg(p.twL + (q - 1) * LA + t + NTS * u);
                    w[2 * (u * (RA - 1) + q - 1)] = x.x;
                    w[2 * (u * (RA - 1) + q - 1) + 1] = x.y;
                }
#pragma unroll
            for (int q = 1; q < RB; q++) {
                const float2 x = __ldg(p.twL + (RA - 1) * LA + (q - 1) * LB + t % LB);
                w2[2 * (q - 1)] = x.x;
                w2[2 * (q - 1) + 1] = x.y;
            }
            tmem_st32(ttw, w);
            tmem_st32(ttw + 32, w2);
            tmem_wait_st();
        }
        long long wcur = -1, nextb = 0;
        int ready_g = -1;
        auto wait_ready = [&](int j) {       // leader: returns once the group of my job j is complete
            const int g = (y + j * ny) >> p.lgGS;
            if (g == ready_g) return;
            if (!(pf_g == g && pf_val >= a_full)) wait_counter(p.a_done + g, a_full, p.err);
            fence_acquire_task();
            ready_g = g;
        };
        auto prefetch_ready = [&](int j) {
            if (j < nbj) {
                const int g = (y + j * ny) >> p.lgGS;
                if (g != ready_g) { pf_g = g; pf_val = ld_relaxed_u32(p.a_done + g); }
            }
        };
        // leader: bulk copy of the G rows of ring position zp into row buffer b (they are adjacent rows of one spectrum)
        auto issue_rows = [&](int b, int zp) {
            asm volatile("fence.proxy.async.global;" ::: "memory");   // the producers' stores -> this copy's reads
            mbar_expect_tx(&s_full[b], (uint32_t)SH::ROW_BYTES);
            bulk_g2s(rowbuf + (size_t)b * G * L, p.Z + (size_t)zp * (N1 * L) + (size_t)(rg * G) * L, (uint32_t)SH::ROW_BYTES, &s_full[b]);
        };
        if (tid == 0 && nbj > 0) {
            prefetch_ready(0);
            wait_ready(0);
            issue_rows(0, zpos);
            prefetch_ready(1);
        }
        gsync<2, NT>();
        for (int bi = 0; bi < nbj; bi++) {
            const int b = bi & 1;
            float4* const buf = rowbuf + (size_t)b * G * L;
            if (m >= nextb) {   // new accumulation window
                if (wcur >= 0) { sink.flush(st, row, t, wcur); sink.begin(st); }
                wcur = (p.c0 + m) / p.M;
                nextb = (wcur + 1) * p.M - p.c0;
            }
            // ---------------- stage a, in place in the landed rows
            float twa[32];
            tmem_ld32(ttw, twa);
            mbar_wait(&s_full[b], (bi >> 1) & 1);
            cpx v[16 / RA][RA];
#pragma unroll
            for (int u = 0; u < 16 / RA; u++)
#pragma unroll
                for (int r = 0; r < RA; r++) v[u][r] = f4_to_cpx(buf[slot * L + t + NTS * u + r * LA]);
            tmem_wait_ld();
            __syncwarp();   // the swizzled stores below land on positions other lanes of this warp have just read
#pragma unroll
            for (int u = 0; u < 16 / RA; u++) {
                const int ja = t + NTS * u;
                const int aja = slot * L + (ja ^ ((ja / 16) & 7));
                dft<RA>(v[u]);
                buf[aja] = cpx_to_f4(v[u][0]);
#pragma unroll
                for (int q = 1; q < RA; q++)
                    buf[aja + q * LA] = cpx_to_f4(cmul(v[u][q], twa[2 * (u * (RA - 1) + q - 1)], twa[2 * (u * (RA - 1) + q - 1) + 1]));
            }
            // the rows are in shared memory: their ring lines are dead (drop them from the L2 instead of letting them
            // be written back) and the producers may reuse the slot
            {
                const float4* zrow = p.Z + (size_t)zpos * (N1 * L) + (size_t)row * L;
#pragma unroll
                for (int i = 0; i < (L * 16) / (NTS * 128); i++)
                    asm volatile("discard.global.L2 [%0], 128;" ::"l"(zrow + (t + NTS * i) * 8) : "memory");
            }
            int zn = zpos + zstride;
            if (zn >= RS) zn -= RS;
            if (tid == 0) {
                red_release_u32(p.b_done + (m >> p.lgGS), (unsigned)G);
                if (bi + 1 < nbj) { wait_ready(bi + 1); prefetch_ready(bi + 2); }
            }
            gsync<2, NT>();
            // every thread is past stage c of the previous job: its buffer takes the next job's rows
            if (tid == 0 && bi + 1 < nbj) issue_rows(b ^ 1, zn);
            // ---------------- stage b (in place per thread), stage c, Stokes into tensor memory
            {
                float twb[32];
                tmem_ld32(ttw + 32, twb);
                cpx w[RB];
#pragma unroll
                for (int r = 0; r < RB; r++) w[r] = f4_to_cpx(buf[addr_b(r)]);
                dft<RB>(w);
                tmem_wait_ld();
                buf[addr_b(0)] = cpx_to_f4(w[0]);
#pragma unroll
                for (int q = 1; q < RB; q++) buf[addr_b(q)] = cpx_to_f4(cmul(w[q], twb[2 * (q - 1)], twb[2 * (q - 1) + 1]));
            }
            __syncwarp();   // stage c reads what its own half-warp wrote
            {
                float a0[32];
                sink.preload(st, a0);
                cpx w[RC];
#pragma unroll
                for (int r = 0; r < RC; r++) w[r] = f4_to_cpx(buf[addr_c(r)]);
                dft<RC>(w);
                sink.put16_preloaded(st, a0, w);
            }
            m += ny;
            zpos = zn;
        }
        if (wcur >= 0) sink.flush(st, row, t, wcur);
        tmem_wait_st();
    }

    // ================= both groups: leave together; the last CTA out resets the launch's counters
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("griddepcontrol.wait;" ::: "memory");
    if (gtid == 0) {
        __threadfence();
        s_last = (atomicAdd(p.role + 3, 1u) == gridDim.x - 1);
    }
    __syncthreads();
    if (s_last) {
        __threadfence();
        for (int i = gtid; i < ngroups; i += NTC) { p.a_done[i] = 0u; p.b_done[i] = 0u; }
        for (int i = gtid; i < kFusedRoleWords; i += NTC) p.role[i] = 0u;
    }
    if (gtid < 32) {
#pragma unroll
        for (int i = 0; i < NSETS; i++)
            asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(*(volatile uint32_t*)&s_tmem[i]), "n"(128) : "memory");
    }
}

}  // namespace spk
