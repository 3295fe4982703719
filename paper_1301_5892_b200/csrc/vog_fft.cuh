// vog_fft.cuh -- in-register radix butterflies and the shared-memory line-FFT plan used by the
// fused advection kernels (sm_100a).  Product code; shares nothing with oracle/.
//
// A "complex line" packs TWO real periodic lines of length N as z = u_A + i u_B (two-for-one:
// the circulant matrices of P:98-100 are real, so one complex FFT serves two lines).  The
// transform is decimation-in-frequency forward / decimation-in-time inverse, in place, so the
// spectrum stays in digit-reversed order and no reordering pass exists: the symbol multiply
// happens in registers between the last forward pass and the first inverse pass.
#pragma once
#include <cuda_runtime.h>

namespace vog {

// ---------------------------------------------------------------------------------------------
// compile-time roots of unity of order 32 (enough for radix <= 32)
__host__ __device__ constexpr double cos32(int k)
{
    // cos(2 pi k / 32), k in [0, 32)
    constexpr double c[9] = {1.0, 0.9807852804032304, 0.9238795325112867, 0.8314696123025452,
                             0.7071067811865476, 0.5555702330196023, 0.38268343236508984,
                             0.19509032201612833, 0.0};
    k &= 31;
    if (k > 16) k = 32 - k;          // cos is even
    return k <= 8 ? c[k] : -c[16 - k];
}
__host__ __device__ constexpr double sin32(int k) { return cos32(k - 8); }

__host__ __device__ constexpr int brev(int q, int R)
{
    int r = 0;
    for (int b = 1; b < R; b <<= 1) { r = (r << 1) | (q & 1); q >>= 1; }
    return r;
}
__host__ __device__ constexpr int ilog2(int n) { int l = 0; while ((1 << l) < n) ++l; return l; }

// Complex arithmetic on packed fp32 pairs (sm_100 FADD2/FMUL2/FFMA2: the same 128 fp32 lanes/cycle/SM as
// the scalar forms but half the issue slots; operand swap / negate / broadcast are instruction modifiers,
// so conj() and multiplication by +-i cost nothing).  Results are bit-identical to the scalar forms.
__device__ __forceinline__ float fneg(float x) { return __int_as_float(__float_as_int(x) ^ 0x80000000); }  // ALU pipe
__device__ __forceinline__ float2 cadd(float2 a, float2 b) { return __fadd2_rn(a, b); }
__device__ __forceinline__ float2 csub(float2 a, float2 b) { return __fadd2_rn(a, make_float2(-b.x, -b.y)); }
// a * b = a b.x + i (a b.y):  FMUL2 by the broadcast scalar b.y, then FFMA2 by the broadcast scalar b.x with the
// product swapped and half-negated as an operand modifier (-R.F32x2.LO_HI.NP): two instructions, no moves.
__device__ __forceinline__ float2 cmul(float2 a, float2 b)
{
    const float2 t = __fmul2_rn(a, make_float2(b.y, b.y));
    return __ffma2_rn(a, make_float2(b.x, b.x), make_float2(-t.y, t.x));
}
// a * conj(b) = a b.x - i (a b.y)
__device__ __forceinline__ float2 cmulc(float2 a, float2 b)
{
    const float2 t = __fmul2_rn(a, make_float2(b.y, b.y));
    return __ffma2_rn(a, make_float2(b.x, b.x), make_float2(t.y, -t.x));
}

// multiply by the compile-time root e^{-/+ 2 pi i K / R} (forward: minus; INV: plus)
template <int K, int R, bool INV>
__device__ __forceinline__ float2 mul_root(float2 d)
{
    constexpr int k32 = (K * (32 / R)) & 31;
    if constexpr (k32 == 0) return d;
    else if constexpr (k32 == 8) return INV ? make_float2(-d.y, d.x) : make_float2(d.y, -d.x);
    else if constexpr (k32 == 16) return make_float2(-d.x, -d.y);
    else if constexpr (k32 == 24) return INV ? make_float2(d.y, -d.x) : make_float2(-d.y, d.x);
    else {
        constexpr float c = (float)cos32(k32);
        constexpr float s = INV ? (float)sin32(k32) : -(float)sin32(k32);
        // d (c + i s) = d c + i (d s): both constants are broadcast immediates, the swap and the half negation
        // of the first product are operand modifiers of the FFMA2 -- two instructions, no constant pairs to build
        const float2 t = __fmul2_rn(d, make_float2(s, s));
        return __ffma2_rn(d, make_float2(c, c), make_float2(-t.y, t.x));
    }
}

// x[(K+H)*S] *= root^K for K = 0..H-1, K a compile-time constant in each instance
template <int K, int H, int R, int S, bool INV>
struct RootLoop {
    static __device__ __forceinline__ void run(float2* x)
    {
        x[(K + H) * S] = mul_root<K, R, INV>(x[(K + H) * S]);
        if constexpr (K + 1 < H) RootLoop<K + 1, H, R, S, INV>::run(x);
    }
};

// Forward DFT of x[0], x[S], .., x[(R-1)S] in registers, decimation in frequency:
// on exit X[q] sits at x[brev(q,R)*S].
template <int R, int S>
__device__ __forceinline__ void dft_dif(float2* x)
{
    if constexpr (R > 1) {
        constexpr int H = R / 2;
#pragma unroll
        for (int k = 0; k < H; ++k) {
            float2 a = x[k * S], b = x[(k + H) * S];
            x[k * S] = cadd(a, b);
            x[(k + H) * S] = csub(a, b);
        }
        RootLoop<0, H, R, S, false>::run(x);   // twiddles on the odd half (compile-time roots)
        dft_dif<H, S>(x);
        dft_dif<H, S>(x + H * S);
    }
}

// Unnormalised inverse DFT, decimation in time: input X[q] at x[brev(q,R)*S], output natural.
template <int R, int S>
__device__ __forceinline__ void idft_dit(float2* x)
{
    if constexpr (R > 1) {
        constexpr int H = R / 2;
        idft_dit<H, S>(x);
        idft_dit<H, S>(x + H * S);
        RootLoop<0, H, R, S, true>::run(x);
#pragma unroll
        for (int k = 0; k < H; ++k) {
            float2 a = x[k * S], b = x[(k + H) * S];
            x[k * S] = cadd(a, b);
            x[(k + H) * S] = csub(a, b);
        }
    }
}

// ---------------------------------------------------------------------------------------------
// Radix plan per line length: N = R1 * 16 (two passes) or N = R1 * R2 * 16 (three passes).
// The last radix is always 16 so the symbol stage holds 2 x 16 complex values per thread.
template <int N> struct Radix;
template <> struct Radix<64>    { static constexpr int P = 2, R1 = 4,  R2 = 1;  };
template <> struct Radix<128>   { static constexpr int P = 2, R1 = 8,  R2 = 1;  };
template <> struct Radix<256>   { static constexpr int P = 2, R1 = 16, R2 = 1;  };
template <> struct Radix<512>   { static constexpr int P = 2, R1 = 32, R2 = 1;  };
template <> struct Radix<1024>  { static constexpr int P = 3, R1 = 4,  R2 = 16; };
template <> struct Radix<2048>  { static constexpr int P = 3, R1 = 8,  R2 = 16; };
template <> struct Radix<4096>  { static constexpr int P = 3, R1 = 16, R2 = 16; };
template <> struct Radix<8192>  { static constexpr int P = 3, R1 = 32, R2 = 16; };
template <> struct Radix<16384> { static constexpr int P = 3, R1 = 32, R2 = 32; };
constexpr int RL = 16;   // last radix

// shared-memory position padding: one float2 of pad per 16 keeps every pass conflict-free
__device__ __forceinline__ int padp(int p) { return p + (p >> 4); }
__host__ __device__ constexpr int padded_len(int N) { return N + N / 16; }

}  // namespace vog
