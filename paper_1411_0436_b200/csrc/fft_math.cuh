// fft_math.cuh — packed-fp32 complex arithmetic and register radix-2/4/8/16 DFTs for sm_100a.
//
// Every complex value on the hot path is a PAIR of complex numbers that undergo identical
// operations: the X and Y polarisations of one time sample / channel ("dual-
// polarization ... complex-valued samples").  cpx.re = (X.re, Y.re), cpx.im = (X.im, Y.im),
// each half a 64-bit register pair, so one FFMA2/FADD2/FMUL2 (PTX fma/add/mul.rn.f32x2) does
// the work of two scalar instructions in one issue slot.  Twiddles are scalars; ptxas folds the
// {c,c} broadcast into the FFMA2 operand (R.F32 modifier).
//
// DFT convention (reading R5): X[k] = sum_n x[n] exp(-2 pi i n k / R),
// forward, unnormalised.  All dft<R>() leave the outputs in natural order in the same array.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace spk {

typedef unsigned long long u64;

__device__ __forceinline__ u64 pk(float lo, float hi) {
    u64 r; asm("mov.b64 %0, {%1,%2};" : "=l"(r) : "f"(lo), "f"(hi)); return r;
}
__device__ __forceinline__ void upk(u64 a, float& lo, float& hi) {
    asm("mov.b64 {%0,%1}, %2;" : "=f"(lo), "=f"(hi) : "l"(a));
}
__device__ __forceinline__ u64 bc(float c) { return pk(c, c); }
__device__ __forceinline__ u64 add2(u64 a, u64 b) {
    u64 d; asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d;
}
__device__ __forceinline__ u64 sub2(u64 a, u64 b) {
    u64 d; asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d;
}
__device__ __forceinline__ u64 mul2(u64 a, u64 b) {
    u64 d; asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d;
}
__device__ __forceinline__ u64 fma2(u64 a, u64 b, u64 c) {
    u64 d; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c)); return d;
}

struct cpx { u64 re, im; };

__device__ __forceinline__ cpx cadd(cpx a, cpx b) { return {add2(a.re, b.re), add2(a.im, b.im)}; }
__device__ __forceinline__ cpx csub(cpx a, cpx b) { return {sub2(a.re, b.re), sub2(a.im, b.im)}; }
// a * (c + i s): 2 FMUL2 + 2 FFMA2
__device__ __forceinline__ cpx cmul(cpx a, float c, float s) {
    cpx r;
    r.re = fma2(a.im, bc(-s), mul2(a.re, bc(c)));
    r.im = fma2(a.im, bc(c), mul2(a.re, bc(s)));
    return r;
}
// a * (-i) = (im, -re)
__device__ __forceinline__ cpx cmul_mi(cpx a) { return {a.im, sub2(0ull, a.re)}; }

template <int R> __device__ __forceinline__ void dft(cpx* v);

template <> __device__ __forceinline__ void dft<1>(cpx*) {}

template <> __device__ __forceinline__ void dft<2>(cpx* v) {
    cpx a = v[0], b = v[1];
    v[0] = cadd(a, b);
    v[1] = csub(a, b);
}

// radix-4, W4 = -i:  X1 = (a0-a2) - i(a1-a3),  X3 = (a0-a2) + i(a1-a3)
__device__ __forceinline__ void dft4(cpx& a0, cpx& a1, cpx& a2, cpx& a3) {
    cpx t0 = cadd(a0, a2), t1 = csub(a0, a2), t2 = cadd(a1, a3), d = csub(a1, a3);
    a0 = cadd(t0, t2);
    a2 = csub(t0, t2);
    a1 = {add2(t1.re, d.im), sub2(t1.im, d.re)};
    a3 = {sub2(t1.re, d.im), add2(t1.im, d.re)};
}
template <> __device__ __forceinline__ void dft<4>(cpx* v) { dft4(v[0], v[1], v[2], v[3]); }

#define SPK_SQRT1_2 0.70710678118654752440f
#define SPK_COS_PI_8 0.92387953251128675613f
#define SPK_SIN_PI_8 0.38268343236508977173f

// radix-8 decimation in frequency: u_i = v_i + v_{i+4}, w_i = (v_i - v_{i+4}) W8^i,
// X[2k] = DFT4(u)[k], X[2k+1] = DFT4(w)[k]
template <> __device__ __forceinline__ void dft<8>(cpx* v) {
    cpx u0 = cadd(v[0], v[4]), u1 = cadd(v[1], v[5]), u2 = cadd(v[2], v[6]), u3 = cadd(v[3], v[7]);
    cpx w0 = csub(v[0], v[4]), d1 = csub(v[1], v[5]), d2 = csub(v[2], v[6]), d3 = csub(v[3], v[7]);
    const u64 h = bc(SPK_SQRT1_2);
    // W8^1 = (1-i)/sqrt2: (re+im, im-re)/sqrt2 ; W8^2 = -i ; W8^3 = (-1-i)/sqrt2: (im-re, -re-im)/sqrt2
    cpx w1 = {mul2(add2(d1.re, d1.im), h), mul2(sub2(d1.im, d1.re), h)};
    cpx w2 = {d2.im, sub2(0ull, d2.re)};
    cpx w3 = {mul2(sub2(d3.im, d3.re), h), mul2(add2(d3.re, d3.im), bc(-SPK_SQRT1_2))};
    dft4(u0, u1, u2, u3);
    dft4(w0, w1, w2, w3);
    v[0] = u0; v[2] = u1; v[4] = u2; v[6] = u3;
    v[1] = w0; v[3] = w1; v[5] = w2; v[7] = w3;
}

// radix-16 as 4 x 4 (n = 4 n1 + j, k = q1 + 4 q2): DFT4 over n1 for each j, twiddle W16^{j q1},
// DFT4 over j for each q1.
template <> __device__ __forceinline__ void dft<16>(cpx* v) {
    dft4(v[0], v[4], v[8], v[12]);   // j=0 -> q1 in slots 0,4,8,12
    dft4(v[1], v[5], v[9], v[13]);   // j=1
    dft4(v[2], v[6], v[10], v[14]);  // j=2
    dft4(v[3], v[7], v[11], v[15]);  // j=3
    // slot 4*q1 + j holds u^(j)[q1]; multiply by W16^{j*q1}, W16^e = (cos(pi e/8), -sin(pi e/8))
    const float c1 = SPK_COS_PI_8, s1 = SPK_SIN_PI_8, h = SPK_SQRT1_2;
    v[5] = cmul(v[5], c1, -s1);    // q1=1,j=1: e=1
    v[6] = cmul(v[6], h, -h);      // q1=1,j=2: e=2
    v[7] = cmul(v[7], s1, -c1);    // q1=1,j=3: e=3
    v[9] = cmul(v[9], h, -h);      // q1=2,j=1: e=2
    v[10] = cmul_mi(v[10]);        // q1=2,j=2: e=4
    v[11] = cmul(v[11], -h, -h);   // q1=2,j=3: e=6
    v[13] = cmul(v[13], s1, -c1);  // q1=3,j=1: e=3
    v[14] = cmul(v[14], -h, -h);   // q1=3,j=2: e=6
    v[15] = cmul(v[15], -c1, s1);  // q1=3,j=3: e=9
    dft4(v[0], v[1], v[2], v[3]);      // q1=0 -> X[0+4 q2] in slots 0..3
    dft4(v[4], v[5], v[6], v[7]);      // q1=1 -> X[1+4 q2]
    dft4(v[8], v[9], v[10], v[11]);    // q1=2
    dft4(v[12], v[13], v[14], v[15]);  // q1=3
    // slot 4*q1 + q2 holds X[q1 + 4 q2]: transpose the 4x4 index to natural order
    cpx t;
#define SPK_SWAP(a, b) t = v[a]; v[a] = v[b]; v[b] = t;
    SPK_SWAP(1, 4) SPK_SWAP(2, 8) SPK_SWAP(3, 12) SPK_SWAP(6, 9) SPK_SWAP(7, 13) SPK_SWAP(11, 14)
#undef SPK_SWAP
}

// ---- exact int8 -> fp32 unpack (reading R13).
// byte b (two's complement) -> float(b), exact for all 256 values: flip the sign bit so the byte
// is b+128 unsigned, drop it into the low mantissa byte of 2^23 (0x4B000000) and subtract
// 2^23+128.  PRMT + FADD per component (the conversion instruction I2F runs at a quarter rate).
__device__ __forceinline__ void unpack4(uint32_t w, float& b0, float& b1, float& b2, float& b3) {
    const uint32_t u = w ^ 0x80808080u;
    b0 = __uint_as_float(__byte_perm(u, 0x4B000000u, 0x7440)) - 8388736.0f;
    b1 = __uint_as_float(__byte_perm(u, 0x4B000000u, 0x7441)) - 8388736.0f;
    b2 = __uint_as_float(__byte_perm(u, 0x4B000000u, 0x7442)) - 8388736.0f;
    b3 = __uint_as_float(__byte_perm(u, 0x4B000000u, 0x7443)) - 8388736.0f;
}


// ---- bulk asynchronous copy global -> shared (cp.async.bulk, SASS UBLKCP) completing on an mbarrier.
// One elected thread issues the copy; every consumer thread waits on the barrier phase.
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "WAIT_%=:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra DONE_%=;\n\t"
        "bra WAIT_%=;\n\t"
        "DONE_%=:\n\t}"
        ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
// size: multiple of 16 bytes; src and dst 16-byte aligned
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}

}  // namespace spk
