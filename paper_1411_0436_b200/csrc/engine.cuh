// engine.cuh — the in-CTA FFT engine and the front ends / sinks that make the three hot kernels:
//   single : unpack + PFB FIR + N-point FFT + Stokes + accumulate            (N <= 4096)
//   pass A : unpack + PFB FIR + N1-point column FFTs + W_N twiddle -> Z (L2)  (four-step, N > 4096)
//   pass B : Z -> N2-point row FFTs + Stokes + accumulate
// PAPER.md:87-96 (section 4, steps 2-5) is the chain; the paper ran it as separate kernels around a
// cuFFT call on a Kepler card — here the stages are fused so a spectrum never
// reaches HBM (BASELINE.json north_star items a-c).
//
// Engine: in-place decimation-in-frequency FFT of length L = RA*RB*RC over an array A[0..L):
//   stage a: items ja < LA=L/RA : v[r]=A[ja+r*LA]; DFT_RA; v[q]*=W_L^{ja q}; A[ja+q*LA]=v[q]
//   stage b: items (qa,jb<LB=LA/RB): v[r]=A[qa*LA+jb+r*LB]; DFT_RB; v[q]*=W_LA^{jb q}; in place
//   stage c: items (qa,qb)        : v[r]=A[qa*LA+qb*LB+r]; DFT_RC
// Output frequency k = qa + RA*(qb + RB*qc) sits at position p = qa*LA + qb*LB + qc (digit
// reversal); accumulators are kept in position order and un-permuted once at read-out.
// Stage a reads straight from the front end (global memory), the last stage feeds the sink from
// registers; only the exchanges between stages touch shared memory.
#pragma once
#include "fft_math.cuh"

namespace spk {

template <int L_, int RA_, int RB_, int RC_>
struct Plan {
    static constexpr int L = L_, RA = RA_, RB = RB_, RC = RC_;
    static constexpr int NST = (RB_ == 1) ? 1 : ((RC_ == 1) ? 2 : 3);
    static constexpr int LA = L_ / RA_;
    static constexpr int LB = LA / RB_;
    static constexpr int NTS = L_ / 16;  // threads per FFT slot; each thread owns 16 points
    static constexpr int RLAST = (NST == 1) ? RA_ : ((NST == 2) ? RB_ : RC_);
    static_assert(RA_ * RB_ * RC_ == L_, "radices must multiply to L");
    static_assert(L_ >= 16 && RA_ <= 16 && RB_ <= 16 && RC_ <= 16, "16 points per thread");
};

__device__ __forceinline__ float4 cpx_to_f4(cpx v) {
    float a, b, c, d;
    upk(v.re, a, b);
    upk(v.im, c, d);
    return make_float4(a, b, c, d);
}
__device__ __forceinline__ cpx f4_to_cpx(float4 z) { return {pk(z.x, z.y), pk(z.z, z.w)}; }

// ---- input view: the virtual concatenation  history ++ new input
struct InputView {
    const uint8_t* hist;  // nhist blocks carried from earlier calls
    const uint8_t* in;    // this call's samples
    int nhist;
};

// one time sample (2*P bytes) of block blk, branch n, as raw bits
template <int P>
__device__ __forceinline__ uint32_t fetch_raw(const InputView& v, long long blk, int n, int N) {
    const uint8_t* base = (blk < v.nhist) ? v.hist + (size_t)blk * N * (2 * P)
                                          : v.in + (size_t)(blk - v.nhist) * N * (2 * P);
    if (P == 2) return __ldg((const uint32_t*)base + n);
    return __ldg((const uint16_t*)base + n);
}
template <int P>
__device__ __forceinline__ cpx unpack_cpx(uint32_t w) {
    if (P == 2) {  // bytes [Xre, Xim, Yre, Yim]: the two magic-number subtractions run as FADD2 on (X,Y) pairs
        const uint32_t u = w ^ 0x80808080u;
        const float f0 = __uint_as_float(__byte_perm(u, 0x4B000000u, 0x7440));
        const float f1 = __uint_as_float(__byte_perm(u, 0x4B000000u, 0x7441));
        const float f2 = __uint_as_float(__byte_perm(u, 0x4B000000u, 0x7442));
        const float f3 = __uint_as_float(__byte_perm(u, 0x4B000000u, 0x7443));
        const u64 k = bc(8388736.0f);
        return {sub2(pk(f0, f2), k), sub2(pk(f1, f3), k)};
    }
    float b0, b1, b2, b3;
    unpack4(w, b0, b1, b2, b3);
    return {pk(b0, 0.f), pk(b1, 0.f)};            // bytes [re, im]
}
template <int P>
__device__ __forceinline__ cpx load_raw(const InputView& v, long long blk, int n, int N) {
    return unpack_cpx<P>(fetch_raw<P>(v, blk, n, N));
}

// front end for `single` and `pass A`: element e of spectrum m is branch n = e*stride + off
template <int MODE_PFB, int P, int WIN = 1>
struct FrontRaw {
    InputView view;
    const float* h;  // T*N coefficients (PFB) / N window values (FFT mode, WIN=1; unused when WIN=0)
    int N, T, stride;
    long long m0;    // spectrum index (in the view) of this launch's job 0
    // bulk staging (direct-FFT mode, stride 1): one spectrum's raw block is N*2P contiguous bytes
    static constexpr bool kBulk = (MODE_PFB == 0);
    static constexpr int kElemBytes = 2 * P;
    __device__ __forceinline__ const void* src(long long job, int) const {
        const long long blk = m0 + job;
        return (blk < view.nhist) ? view.hist + (size_t)blk * N * (2 * P)
                                  : view.in + (size_t)(blk - view.nhist) * N * (2 * P);
    }
    __device__ __forceinline__ cpx decode(const void* x, int e, int = 0) const {
        const uint32_t w = (P == 2) ? ((const uint32_t*)x)[e] : (uint32_t)((const uint16_t*)x)[e];
        cpx v = unpack_cpx<P>(w);
        if (WIN) {
            const u64 c = bc(__ldg(h + e));
            v.re = mul2(v.re, c);
            v.im = mul2(v.im, c);
        }
        return v;
    }
    __device__ __forceinline__ int off(int slot_id) const { return stride == 1 ? 0 : slot_id; }
    // test hook (k_engine DUMP): element e of spectrum `job` as the caller's [job][n][re,im per pol]
    __device__ __forceinline__ void dump_put(float* dump, long long job, int e, int off_, cpx v) const {
        const size_t o = (size_t)job * N + (size_t)e * stride + off_;
        const float4 z = cpx_to_f4(v);   // (Xre, Yre, Xim, Yim)
        if (P == 2) ((float4*)dump)[o] = make_float4(z.x, z.z, z.y, z.w);
        else ((float2*)dump)[o] = make_float2(z.x, z.z);
    }
    __device__ __forceinline__ cpx load(long long job, int e, int off_) const {
        const int n = e * stride + off_;
        const long long m = m0 + job;
        if (MODE_PFB) {
            // y[m][n] = sum_t h[tN+n] x[(m+t)N+n]
            u64 re = 0ull, im = 0ull;
            for (int t = 0; t < T; t++) {
                cpx x = load_raw<P>(view, m + t, n, N);
                const u64 c = bc(__ldg(h + (size_t)t * N + n));
                re = fma2(x.re, c, re);
                im = fma2(x.im, c, im);
            }
            return {re, im};
        } else {
            cpx x = load_raw<P>(view, m, n, N);
            if (WIN) {
                const u64 c = bc(__ldg(h + n));
                x.re = mul2(x.re, c);
                x.im = mul2(x.im, c);
            }
            return x;
        }
    }
};

// Direct-FFT front end for N = 2 L with NO intermediate: slot variant r (0 / 1) computes the even / odd channels of the
// N-point transform as ONE L-point transform of  x[n] + x[n+L]  /  (x[n] - x[n+L]) W_N^n  (the first radix-2
// decimation-in-frequency layer), each from the whole raw block.  The unpack is done twice, in exchange
// the 16 B per sample four-step intermediate and its cross-SM hand-over disappear (N = 8192: one k_engine launch).
template <int WIN>
struct FrontRawR2 {
    InputView view;
    const float2* twN;   // W_N^e
    const float* h;      // WIN: window over N
    int N, L;            // N = 2 L
    long long m0;
    int stride = 1;      // (dump_put)
    static constexpr bool kBulk = true;
    static constexpr int kElemBytes = 8;   // element e of the staged block = samples e and e + L
    __device__ __forceinline__ const void* src(long long job, int) const {
        const long long blk = m0 + job;
        return (blk < view.nhist) ? view.hist + (size_t)blk * N * 4 : view.in + (size_t)(blk - view.nhist) * N * 4;
    }
    __device__ __forceinline__ int off(int variant) const { return variant; }
    __device__ __forceinline__ cpx decode(const void* x, int e, int r) const {
        cpx a = unpack_cpx<2>(((const uint32_t*)x)[e]), b = unpack_cpx<2>(((const uint32_t*)x)[e + L]);
        if (WIN) {
            const u64 ca = bc(__ldg(h + e)), cb = bc(__ldg(h + e + L));
            a = {mul2(a.re, ca), mul2(a.im, ca)};
            b = {mul2(b.re, cb), mul2(b.im, cb)};
        }
        if (r == 0) return cadd(a, b);
        const float2 w = __ldg(twN + e);
        return cmul(csub(a, b), w.x, w.y);
    }
    __device__ __forceinline__ cpx load(long long job, int e, int r) const { return decode(src(job, r), e, r); }
    // test hook: what this front end hands to the L-point transform, [job][r][e]: r = 0 the sums x[e] + x[e+L]
    // (exact integers), r = 1 the twiddled differences
    __device__ __forceinline__ void dump_put(float* dump, long long job, int e, int r, cpx v) const {
        const float4 z = cpx_to_f4(v);
        ((float4*)dump)[(size_t)job * N + (size_t)r * L + e] = make_float4(z.x, z.z, z.y, z.w);
    }
};

// front end for `pass B`: row `slot_id` of the intermediate Z[m][row][n2] (float4 = Xre,Yre,Xim,Yim)
struct FrontZ {
    const float4* Z;
    int N, N2;
    static constexpr bool kBulk = true;   // one row of one spectrum is N2*16 contiguous bytes
    static constexpr int kElemBytes = 16;
    __device__ __forceinline__ const void* src(long long m, int row) const {
        return Z + (size_t)m * N + (size_t)row * N2;
    }
    __device__ __forceinline__ cpx decode(const void* x, int e, int = 0) const { return f4_to_cpx(((const float4*)x)[e]); }
    __device__ __forceinline__ int off(int slot_id) const { return slot_id; }
    __device__ __forceinline__ void dump_put(float*, long long, int, int, cpx) const {}
    __device__ __forceinline__ cpx load(long long m, int e, int row) const {
        const float4 z = Z[(size_t)m * N + (size_t)row * N2 + e];
        return {pk(z.x, z.y), pk(z.z, z.w)};
    }
};

// front end for `pass A` behind the stand-alone FIR kernel (k_fir8, passa_pfb.cuh): element e of column
// `off` of the filtered spectrum Y[m][n] (float4 = Xre,Yre,Xim,Yim), n = e*stride + off
struct FrontY {
    const float4* Y;
    int N, stride;
    static constexpr bool kBulk = false;
    static constexpr int kElemBytes = 16;
    __device__ __forceinline__ const void* src(long long, int) const { return nullptr; }
    __device__ __forceinline__ cpx decode(const void*, int, int = 0) const { return {0ull, 0ull}; }
    __device__ __forceinline__ int off(int slot_id) const { return slot_id; }
    __device__ __forceinline__ void dump_put(float*, long long, int, int, cpx) const {}
    __device__ __forceinline__ cpx load(long long m, int e, int off_) const {
        return f4_to_cpx(__ldcg(Y + (size_t)m * N + (size_t)e * stride + off_));
    }
};

// accumulator update without a return value: one vector reduction at the L2 (RED.E.ADD.F32x4), nothing comes back
// to the SM (atomicAdd(float4*) compiles to ATOMG, whose result the thread then waits for)
__device__ __forceinline__ void red_add_f4(float4* p, float a, float b, float c, float d) {
    asm volatile("red.relaxed.gpu.global.add.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(p), "f"(a), "f"(b), "f"(c), "f"(d) : "memory");
}
__device__ __forceinline__ void red_add_f1(float* p, float a) {
    asm volatile("red.relaxed.gpu.global.add.f32 [%0], %1;" ::"l"(p), "f"(a) : "memory");
}

// ---- sinks
// The last engine stage hands each sink the 16 outputs of one radix-16 butterfly at once:
//   put16(state, m, off, i, k0, ks, v): v[q] is the output at engine position p = 16*i + q,
//   frequency k = k0 + ks*q of the L-point transform, spectrum (job) m, column/row offset `off`.
// Stokes detection + accumulation: XX=|X|^2, YY=|Y|^2, Re(X conj Y), Im(X conj Y)
template <int P>
struct SinkStokes {
    float* ring;     // nring accumulators, each [position][S] fp32, S = 4 (P=2) or 1 (P=1)
    size_t stride;   // floats per accumulator (S*N)
    int nring;       // accumulation window w lives in ring slot w % nring
    int slot_len;    // positions per slot (L)
    int rows_mode;   // 1: slot_id selects a row of the accumulator (pass B); 0: all slots share it
    static constexpr bool kAccumulates = true;
    static constexpr bool kTmem = false;
    struct State {
        u64 pw[16];
        float cr[16], ci[16];
    };
    __device__ __forceinline__ void init(State&, uint32_t, int = 64) const {}
    __device__ __forceinline__ void begin(State& s) const {
#pragma unroll
        for (int i = 0; i < 16; i++) { s.pw[i] = 0ull; s.cr[i] = 0.f; s.ci[i] = 0.f; }
    }
    __device__ __forceinline__ void put16(State& s, long long, int, int, int, int, const cpx* v) const {
#pragma unroll
        for (int q = 0; q < 16; q++) {
            s.pw[q] = fma2(v[q].re, v[q].re, s.pw[q]);
            s.pw[q] = fma2(v[q].im, v[q].im, s.pw[q]);
            if (P == 2) {
                float xr, yr, xi, yi;
                upk(v[q].re, xr, yr);
                upk(v[q].im, xi, yi);
                s.cr[q] = fmaf(xr, yr, fmaf(xi, yi, s.cr[q]));   // Re(X conj Y) = XrYr + XiYi
                s.ci[q] = fmaf(xi, yr, fmaf(-xr, yi, s.ci[q]));  // Im(X conj Y) = XiYr - XrYi
            }
        }
    }
    // add the partial sums of the 16 positions 16*i .. 16*i+15 to window w's accumulator
    __device__ __forceinline__ void flush(State& s, int slot_id, int i, long long w) const {
        float* acc = ring + (size_t)(w % nring) * stride;
        const size_t pos = (rows_mode ? (size_t)slot_id * slot_len : 0) + (size_t)i * 16;
#pragma unroll
        for (int q = 0; q < 16; q++) {
            float xx, yy;
            upk(s.pw[q], xx, yy);
            if (P == 2) red_add_f4((float4*)acc + pos + q, xx, yy, s.cr[q], s.ci[q]);
            else red_add_f1(acc + pos + q, xx);
        }
    }
};

// ---- tensor memory as accumulator storage (sm_100a).  The 4 Stokes sums of the 16 channels a
// thread owns are 64 fp32 words that are touched once per spectrum; kept in registers they cost
// 64 registers per thread and halve the occupancy of the FFT.  TMEM (256 KB per SM, idle here
// because no tensor-core instruction runs) holds them instead: each thread owns 64 columns of its
// own TMEM lane (tcgen05.ld/st .32x32b: thread i of a warp <-> lane 32*(warp%4)+i), read-modify-
// written 32 words at a time around the Stokes FMAs.
__device__ __forceinline__ void tmem_ld32(uint32_t taddr, float* r) {
    uint32_t* u = (uint32_t*)r;
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
        "{%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,"
        "%16,%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31}, [%32];"
        : "=r"(u[0]), "=r"(u[1]), "=r"(u[2]), "=r"(u[3]), "=r"(u[4]), "=r"(u[5]), "=r"(u[6]), "=r"(u[7]),
          "=r"(u[8]), "=r"(u[9]), "=r"(u[10]), "=r"(u[11]), "=r"(u[12]), "=r"(u[13]), "=r"(u[14]), "=r"(u[15]),
          "=r"(u[16]), "=r"(u[17]), "=r"(u[18]), "=r"(u[19]), "=r"(u[20]), "=r"(u[21]), "=r"(u[22]), "=r"(u[23]),
          "=r"(u[24]), "=r"(u[25]), "=r"(u[26]), "=r"(u[27]), "=r"(u[28]), "=r"(u[29]), "=r"(u[30]), "=r"(u[31])
        : "r"(taddr)
        : "memory");
}
__device__ __forceinline__ void tmem_st32(uint32_t taddr, const float* r) {
    const uint32_t* u = (const uint32_t*)r;
    asm volatile(
        "tcgen05.st.sync.aligned.32x32b.x32.b32 [%0], "
        "{%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,"
        "%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31,%32};"
        ::"r"(taddr), "r"(u[0]), "r"(u[1]), "r"(u[2]), "r"(u[3]), "r"(u[4]), "r"(u[5]), "r"(u[6]), "r"(u[7]),
          "r"(u[8]), "r"(u[9]), "r"(u[10]), "r"(u[11]), "r"(u[12]), "r"(u[13]), "r"(u[14]), "r"(u[15]),
          "r"(u[16]), "r"(u[17]), "r"(u[18]), "r"(u[19]), "r"(u[20]), "r"(u[21]), "r"(u[22]), "r"(u[23]),
          "r"(u[24]), "r"(u[25]), "r"(u[26]), "r"(u[27]), "r"(u[28]), "r"(u[29]), "r"(u[30]), "r"(u[31])
        : "memory");
}
__device__ __forceinline__ void tmem_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void tmem_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }
// one warp allocates NCOLS columns (power of two >= 32) for the CTA and publishes the base address
template <int NCOLS>
__device__ __forceinline__ uint32_t tmem_alloc_cta(uint32_t* slot_smem) {
    if (threadIdx.x < 32) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(slot_smem)), "n"(NCOLS) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    return *(volatile uint32_t*)slot_smem;
}
template <int NCOLS>
__device__ __forceinline__ void tmem_free_cta(uint32_t base) {
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (threadIdx.x < 32)
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(base), "n"(NCOLS) : "memory");
}

// The persistent kernels (fused.cuh, fused2.cuh) allocate tensor memory ONLY in blocks of 128 columns, one per set of four
// warps that needs one.  Their CTAs wait for one another, so a CTA blocked in tcgen05.alloc behind a CTA of its own grid
// is a deadlock: with a single 256-column request per CTA, two foreign 128-column allocations (a pass-B launch of another
// handle, say) on either side of the first CTA's block leave 256 free but not contiguous columns once they are gone, and
// the second CTA of the SM never starts (seen once as a 10 s time-out in the soak test).  Requests of one size cannot
// fragment: a free block of 128 always serves the next one.
template <int NSETS>
__device__ __forceinline__ void tmem_alloc_sets(uint32_t* slots_smem) {
    if (threadIdx.x < 32) {
#pragma unroll
        for (int i = 0; i < NSETS; i++)
            asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(slots_smem + i)), "n"(128) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
}
template <int NSETS>
__device__ __forceinline__ void tmem_free_sets(const uint32_t* slots_smem) {
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (threadIdx.x < 32) {
#pragma unroll
        for (int i = 0; i < NSETS; i++)
            asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(*(volatile const uint32_t*)(slots_smem + i)), "n"(128) : "memory");
    }
}

// dual-pol Stokes sink with the accumulators in tensor memory: column 4*q+{0,1,2,3} of the thread's
// lane = XX, YY, Re, Im of its position 16*i+q
struct SinkStokesTmem {
    float* ring;
    size_t stride;
    int nring;
    int slot_len;
    int rows_mode;
    static constexpr bool kAccumulates = true;
    static constexpr bool kTmem = true;
    struct State {
        uint32_t taddr;
    };
    // colstride: columns reserved per set of four warps (64 accumulator words, plus whatever else the
    // kernel keeps in the thread's lane)
    __device__ __forceinline__ void init(State& s, uint32_t tmem_base, int colstride = 64) const {
        const int warp = threadIdx.x >> 5;
        s.taddr = tmem_base + ((uint32_t)((warp & 3) * 32) << 16) + (uint32_t)((warp >> 2) * colstride);
    }
    // the thread's set of four warps owns the 128-column block at `set_base` (tmem_alloc_sets)
    __device__ __forceinline__ void init_set(State& s, uint32_t set_base) const {
        const int warp = threadIdx.x >> 5;
        s.taddr = set_base + ((uint32_t)((warp & 3) * 32) << 16);
    }
    __device__ __forceinline__ void begin(State& s) const {
        float z[32];
#pragma unroll
        for (int i = 0; i < 32; i++) z[i] = 0.f;
        tmem_st32(s.taddr, z);
        tmem_st32(s.taddr + 32, z);
        tmem_wait_st();
    }
    static __device__ __forceinline__ void stokes8(float* a, const cpx* v) {
#pragma unroll
        for (int j = 0; j < 8; j++) {
            const cpx x = v[j];
            u64 pw = pk(a[4 * j], a[4 * j + 1]);
            pw = fma2(x.re, x.re, pw);
            pw = fma2(x.im, x.im, pw);
            upk(pw, a[4 * j], a[4 * j + 1]);
            float xr, yr, xi, yi;
            upk(x.re, xr, yr);
            upk(x.im, xi, yi);
            a[4 * j + 2] = fmaf(xr, yr, fmaf(xi, yi, a[4 * j + 2]));   // Re(X conj Y) = XrYr + XiYi
            a[4 * j + 3] = fmaf(xi, yr, fmaf(-xr, yi, a[4 * j + 3]));  // Im(X conj Y) = XiYr - XrYi
        }
    }
    // The stores of one call are only waited for at the start of the next TMEM access of the thread
    // (next job), so they overlap whatever comes in between.
    __device__ __forceinline__ void put16(State& s, long long, int, int, int, int, const cpx* v) const {
        tmem_wait_st();
#pragma unroll
        for (int hh = 0; hh < 2; hh++) {
            float a[32];
            tmem_ld32(s.taddr + 32 * hh, a);
            tmem_wait_ld();
            stokes8(a, v + 8 * hh);
            tmem_st32(s.taddr + 32 * hh, a);
        }
    }
    // split form: `preload` before the last butterfly, `put16_preloaded` after it
    __device__ __forceinline__ void preload(State& s, float* a0) const {
        tmem_wait_st();
        tmem_ld32(s.taddr, a0);
    }
    __device__ __forceinline__ void put16_preloaded(State& s, float* a0, const cpx* v) const {
        float a1[32];
        tmem_wait_ld();
        tmem_ld32(s.taddr + 32, a1);
        stokes8(a0, v);
        tmem_st32(s.taddr, a0);
        tmem_wait_ld();
        stokes8(a1, v + 8);
        tmem_st32(s.taddr + 32, a1);
    }
    __device__ __forceinline__ void flush(State& s, int slot_id, int i, long long w) const {
        float4* acc = (float4*)(ring + (size_t)(w % nring) * stride);
        const size_t pos = (rows_mode ? (size_t)slot_id * slot_len : 0) + (size_t)i * 16;
        tmem_wait_st();
#pragma unroll
        for (int hh = 0; hh < 2; hh++) {
            float a[32];
            tmem_ld32(s.taddr + 32 * hh, a);
            tmem_wait_ld();
#pragma unroll
            for (int j = 0; j < 8; j++)
                red_add_f4(acc + pos + 8 * hh + j, a[4 * j], a[4 * j + 1], a[4 * j + 2], a[4 * j + 3]);
        }
    }
};

// pass A sink: multiply by the four-step twiddle W_N^{n2 k1} and store Z[m][p1][n2]
struct SinkZ {
    float4* Z;
    const float2* twN;  // W_N^e, e < N
    int N, N2;
    static constexpr bool kAccumulates = false;
    static constexpr bool kTmem = false;
    struct State {};
    __device__ __forceinline__ void init(State&, uint32_t, int = 64) const {}
    __device__ __forceinline__ void begin(State&) const {}
    __device__ __forceinline__ void put16(State&, long long m, int n2, int i, int k0, int ks, const cpx* v) const {
#pragma unroll
        for (int q = 0; q < 16; q++) {
            const int k = k0 + ks * q;
            cpx x = v[q];
            if (k) {
                const float2 w = __ldg(twN + (size_t)n2 * k);
                x = cmul(x, w.x, w.y);
            }
            float a, b, c, d;
            upk(x.re, a, b);
            upk(x.im, c, d);
            Z[(size_t)m * N + (size_t)(16 * i + q) * N2 + n2] = make_float4(a, b, c, d);
        }
    }
    __device__ __forceinline__ void flush(State&, int, int, long long) const {}
};

// ---- job map: which spectra a slot processes
struct JobMap {
    long long njobs;   // spectra in this launch
    int len;           // spectra per slot (runs mode) or per blockIdx.y chunk
    int nslots;        // valid slots (columns / rows / runs x variants)
    int runs_mode;     // 1: slot_id indexes a run of spectra (single); 0: blockIdx.y does
    int nrun;          // runs mode: number of runs; slot_id = variant * nrun + run (variant 0 only unless the front end
                       // splits a spectrum over several slots, FrontRawR2)
    long long c0;      // spectrum count since stream start at job 0 (accumulation windows)
    long long M;       // spectra per accumulation window
    int pdl = 0;       // 1: this launch lets the next launch of the stream start early (accumulating single-kernel plans only;
                       // a pass-A / pass-B launch must NOT: what follows it reads or overwrites its Z)
};


// The kernel.  G FFT slots per CTA, PL::NTS threads each.
//   IL = false ("slot-major"): tid -> slot = tid / NTS, t = tid % NTS; A[p] at slot*L + swz(p)
//   IL = true  ("interleaved", pass A): slot = tid % G, t = tid / G; A[p] at p*G + slot, so that
//        adjacent lanes are adjacent columns n2 (coalesced input rows and Z rows, no bank conflicts)
//   DUMP (test hook for the bit-exact stage tests): stage a writes what the front end delivered (unpacked
//        samples / FIR outputs / windowed samples) to `dump` as [job][n][re,im per pol] and nothing else runs
template <class PL, bool IL, int G, int MINB, class Front, class Sink, bool DUMP = false>
__global__ void __launch_bounds__(PL::NTS * G, MINB)
k_engine(const Front front, const Sink sink, const JobMap jm, const float2* __restrict__ twL, float* __restrict__ dump) {
    constexpr int L = PL::L, RA = PL::RA, RB = PL::RB, RC = PL::RC, NST = PL::NST;
    constexpr int LA = PL::LA, LB = PL::LB, NTS = PL::NTS;
    extern __shared__ float4 smem[];
    // BULK: the next job's input is copied global -> shared by cp.async.bulk while this job computes
    constexpr bool BULK = Front::kBulk && !IL && NST >= 2;
    constexpr int XB = L * Front::kElemBytes;                      // staged bytes per slot
    uint8_t* xbuf = (uint8_t*)(smem + (size_t)G * L);              // [G][XB]
    uint64_t* bar = (uint64_t*)(xbuf + (BULK ? (size_t)G * XB : 0));  // mbarrier, then the TMEM base slot

    const int tid = threadIdx.x;
    const int slot = IL ? (tid % G) : (tid / NTS);
    const int t = IL ? (tid / G) : (tid % NTS);
    const int slot_id = blockIdx.x * G + slot;
    const bool slot_ok = slot_id < jm.nslots;
    const long long j0 = (long long)(jm.runs_mode ? slot_id % jm.nrun : blockIdx.y) * jm.len;
    const long long j1 = (j0 + jm.len < jm.njobs) ? j0 + jm.len : jm.njobs;
    const int off = front.off(jm.runs_mode ? slot_id / jm.nrun : slot_id);
    const int acc_slot = jm.runs_mode ? slot_id / jm.nrun : slot_id;   // which stretch of the accumulator this slot adds to

    // last-stage swizzle of the slot-major layout: RLAST contiguous points per item, so XOR the low
    // bits with the item index to spread a quarter-warp over all banks
    auto addr = [&](int p) -> int {
        if (IL) return p * G + slot;
        constexpr int RL = PL::RLAST;
        const int s = (RL >= 8) ? (p ^ ((p / RL) & 7)) : p;
        return slot * L + s;
    };
    // The same swizzle written out for the slot-major three-stage plans (LA = 256, LB = RB = RC = 16): the 16
    // addresses of a stage become one base + compile-time offsets + one of the 8 values (t & 7) ^ k instead of
    // 16 independent registers per stage (see fused.cuh: ptxas hoists and spills those)
    constexpr bool kExplicit = !IL && (NST == 3) && (PL::RLAST == 16) && (LA % 128 == 0) && (LB == 16) && (RB == 16) && (RC == 16);
    const int c7 = t & 7;
    const int bbase = slot * L + (t >> 4) * LA + (t & 8);
    const int cbase = slot * L + 16 * t;
    auto addr_b = [&](int r) -> int { return bbase + 16 * r + (c7 ^ (r & 7)); };   // == addr((t/16)*LA + t%16 + 16 r)
    auto addr_c = [&](int r) -> int { return cbase + (r & 8) + (c7 ^ (r & 7)); };  // == addr(16 t + r)

    // TMEM accumulators (SinkStokesTmem): 64 columns per warp-quarter set; needs warp-uniform control
    // flow around the tcgen05 instructions, i.e. at least one warp per slot
    // With the TMEM sink the stage twiddles of the thread (the same for every job) are parked in TMEM
    // too: columns 64.. of its lane, one tcgen05.ld per stage instead of up to 30 table loads per job.
    constexpr int TCOLS = (NTS * G > 128) ? 256 : 128;
    constexpr int TWA = (NST >= 2) ? (16 / RA) * (RA - 1) : 0;       // float2 per thread, stage a
    constexpr int TWB = (NST == 3) ? (16 / RB) * (RB - 1) : 0;       // stage b
    static_assert(!Sink::kTmem || NTS >= 32, "TMEM sink: a slot must be at least one warp");
    static_assert(TWA <= 16 && TWB <= 16, "32 words per stage");
    uint32_t tmem_base = 0;
    if (Sink::kTmem) tmem_base = tmem_alloc_cta<TCOLS>((uint32_t*)(bar + 1));
    typename Sink::State st;
    sink.init(st, tmem_base, 128);
    sink.begin(st);
    // Programmatic dependent launch (accumulating single-kernel launches only, spec.cu sets the attribute): the next
    // spec_process call's launch may fill the SM slots this grid's last wave frees one by one.  The two grids share
    // nothing but the accumulators (commutative reductions) and read-only tables; a no-op for ordinary launches.
    if (jm.pdl) asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    uint32_t ttw = 0;
    if (Sink::kTmem) {
        const int warp = tid >> 5;
        ttw = tmem_base + ((uint32_t)((warp & 3) * 32) << 16) + (uint32_t)((warp >> 2) * 128) + 64;
        float w[32];
#pragma unroll
        for (int i = 0; i < 32; i++) w[i] = 0.f;
#pragma unroll
        for (int u = 0; u < 16 / RA; u++)
#pragma unroll
            for (int q = 1; q < RA; q++) {
                if (NST >= 2) {
                    const float2 x = __ldg(twL + (q - 1) * LA + t + NTS * u);
                    w[2 * (u * (RA - 1) + q - 1)] = x.x;
                    w[2 * (u * (RA - 1) + q - 1) + 1] = x.y;
                }
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
                    const float2 x = __ldg(twL + (RA - 1) * LA + (q - 1) * LB + (t + NTS * u) % LB);
                    w2[2 * (u * (RB - 1) + q - 1)] = x.x;
                    w2[2 * (u * (RB - 1) + q - 1) + 1] = x.y;
                }
            tmem_st32(ttw + 32, w2);
        }
        tmem_wait_st();
    }
    // accumulation window of the current job and the job index at which the next window starts:
    // a run that crosses a window boundary flushes its partial sums there and starts over
    long long wcur = (jm.c0 + j0) / jm.M;
    long long nextb = (wcur + 1) * jm.M - jm.c0;
    static_assert(PL::RLAST == 16, "the last stage is always radix 16 (one put16 per thread and job)");
    auto flush_all = [&](long long w) { sink.flush(st, acc_slot, t, w); };

    // thread 0 issues the copies of iteration `it` for every slot of the CTA
    auto issue = [&](int it) {
        uint32_t bytes = 0;
        for (int g = 0; g < G; g++) {
            const int sid = blockIdx.x * G + g;
            const long long gj0 = (long long)(jm.runs_mode ? sid % jm.nrun : blockIdx.y) * jm.len;
            const long long gj1 = (gj0 + jm.len < jm.njobs) ? gj0 + jm.len : jm.njobs;
            if (sid < jm.nslots && gj0 + it < gj1) bytes += XB;
        }
        mbar_expect_tx(bar, bytes);
        for (int g = 0; g < G; g++) {
            const int sid = blockIdx.x * G + g;
            const long long gj0 = (long long)(jm.runs_mode ? sid % jm.nrun : blockIdx.y) * jm.len;
            const long long gj1 = (gj0 + jm.len < jm.njobs) ? gj0 + jm.len : jm.njobs;
            if (sid < jm.nslots && gj0 + it < gj1)
                bulk_g2s(xbuf + (size_t)g * XB, front.src(gj0 + it, front.off(jm.runs_mode ? sid / jm.nrun : sid)), XB, bar);
        }
    };
    if (BULK) {
        if (tid == 0) mbar_init(bar, 1);
        __syncthreads();
        if (tid == 0) issue(0);
    }

    for (int it = 0; it < jm.len; it++) {
        const long long m = j0 + it;
        const bool active = slot_ok && (m < j1);
        if (BULK) mbar_wait(bar, it & 1);
        if (Sink::kAccumulates && !DUMP && active && m == nextb) {
            flush_all(wcur);
            sink.begin(st);
            wcur++;
            nextb += jm.M;
        }
        // ---------------- stage a
        if (active) {
            float twa[32];
            if (Sink::kTmem && NST >= 2) { tmem_ld32(ttw, twa); tmem_wait_ld(); }
#pragma unroll
            for (int u = 0; u < 16 / RA; u++) {
                const int ja = t + NTS * u;
                cpx v[RA];
#pragma unroll
                for (int r = 0; r < RA; r++)
                    v[r] = BULK ? front.decode(xbuf + (size_t)slot * XB, ja + r * LA, off) : front.load(m, ja + r * LA, off);
                if (DUMP) {
#pragma unroll
                    for (int r = 0; r < RA; r++) front.dump_put(dump, m, ja + r * LA, off, v[r]);
                    continue;
                }
                dft<RA>(v);
                if (NST == 1) {
                    sink.put16(st, m, off, ja, 0, 1, v);
                } else {
                    const int aja = addr(ja);
                    smem[aja] = cpx_to_f4(v[0]);
#pragma unroll
                    for (int q = 1; q < RA; q++) {
                        float2 w;
                        if (Sink::kTmem) w = make_float2(twa[2 * (u * (RA - 1) + q - 1)], twa[2 * (u * (RA - 1) + q - 1) + 1]);
                        else w = __ldg(twL + (q - 1) * LA + ja);  // W_L^{ja q}, table [q][ja]
                        smem[kExplicit ? aja + q * LA : addr(ja + q * LA)] = cpx_to_f4(cmul(v[q], w.x, w.y));
                    }
                }
            }
        }
        if (NST >= 2) {
            __syncthreads();
            if (BULK && tid == 0 && it + 1 < jm.len) issue(it + 1);  // the staging buffer is free again
            // ---------------- stage b
            if (active && !DUMP) {
                float twb[32];
                if (Sink::kTmem && NST == 3) { tmem_ld32(ttw + 32, twb); tmem_wait_ld(); }
#pragma unroll
                for (int u = 0; u < 16 / RB; u++) {
                    const int i = t + NTS * u;
                    const int qa = i / LB, jb = i % LB;
                    const int base = qa * LA + jb;
                    cpx v[RB];
#pragma unroll
                    for (int r = 0; r < RB; r++) v[r] = f4_to_cpx(smem[kExplicit ? addr_b(r) : addr(base + r * LB)]);
                    dft<RB>(v);
                    if (NST == 2) {  // LB == 1: i == qa, p = qa*RB + q, k = qa + RA*q
                        sink.put16(st, m, off, i, i, RA, v);
                    } else {
                        smem[kExplicit ? addr_b(0) : addr(base)] = cpx_to_f4(v[0]);
#pragma unroll
                        for (int q = 1; q < RB; q++) {
                            float2 w;
                            if (Sink::kTmem) w = make_float2(twb[2 * (u * (RB - 1) + q - 1)], twb[2 * (u * (RB - 1) + q - 1) + 1]);
                            else w = __ldg(twL + (RA - 1) * LA + (q - 1) * LB + jb);  // W_LA^{jb q}, table [q][jb]
                            smem[kExplicit ? addr_b(q) : addr(base + q * LB)] = cpx_to_f4(cmul(v[q], w.x, w.y));
                        }
                    }
                }
            }
            // three-stage plans: stage c only reads what the same 16 adjacent threads wrote in stage b
            // (one block of LA points), so a warp-level barrier is enough there
            if (NST == 3 && !IL && LB == 16 && RC == 16) __syncwarp();
            else __syncthreads();
        }
        if (NST == 3) {
            // ---------------- stage c
            if (active && !DUMP) {
#pragma unroll
                for (int u = 0; u < 16 / RC; u++) {
                    const int i = t + NTS * u;  // i = qa*RB + qb
                    cpx v[RC];
#pragma unroll
                    for (int r = 0; r < RC; r++) v[r] = f4_to_cpx(smem[kExplicit ? addr_c(r) : addr(i * RC + r)]);
                    dft<RC>(v);
                    const int qa = i / RB, qb = i % RB;
                    sink.put16(st, m, off, i, qa + RA * qb, RA * RB, v);
                }
            }
            __syncthreads();
        }
    }

    if (Sink::kAccumulates && !DUMP && slot_ok && j0 < j1) flush_all(wcur);
    // (a grid that overlapped its predecessor's tail must not COMPLETE before it: whatever follows in the stream, a
    // read-out for one, relies on stream order)
    asm volatile("griddepcontrol.wait;" ::: "memory");
    if (Sink::kTmem) tmem_free_cta<TCOLS>(tmem_base);
}

}  // namespace spk
