// vog_advect_x.cuh -- fused advection kernel for CONTIGUOUS lines (x-direction; SURVEY.md 8(a)
// steps S2-S5, S7).  Product code; shares nothing with oracle/.
//
// A velocity row of N floats is, in its natural memory order, a complex array z_n = u_2n + i u_2n+1
// of M = N/2 float2 (even/odd packing of a real sequence).  One complex FFT of length M, the
// "untangle" U_k = E_k + W_N^k O_k, the multiplication by the eigenvalues lambda_k of the circulant
// interpolation matrix (closed form), the re-tangle and the inverse FFT
// give the advected row in place:
//   * every global and shared access is 128 bit;
//   * the line lives in shared memory as 4N bytes with an XOR swizzle of the 16-byte chunk index
//     (chunk bits 0-2 ^= bits 3-5), which makes the strided radix passes AND the contiguous radix-16
//     middle stage bank-conflict free without padding;
//   * CTAs are persistent and double-buffered: cp.async lands line group g+1 (and its shift records)
//     while group g is transformed; results leave from registers as streaming 128-bit stores.
// Transform structure: decimation in frequency forward / decimation in time inverse, in place,
// spectrum left digit-reversed; M = R1 * [16 *] 16.
#pragma once
#include "vog_fft.cuh"
#include "vog_internal.h"

namespace vog {

// ---- radix plan for the complex length M = N/2
template <int N> struct XPlan;
template <> struct XPlan<64>    { static constexpr int R1 = 2,  R2 = 1;  };
template <> struct XPlan<128>   { static constexpr int R1 = 4,  R2 = 1;  };
template <> struct XPlan<256>   { static constexpr int R1 = 8,  R2 = 1;  };
template <> struct XPlan<512>   { static constexpr int R1 = 16, R2 = 1;  };
template <> struct XPlan<1024>  { static constexpr int R1 = 32, R2 = 1;  };
template <> struct XPlan<2048>  { static constexpr int R1 = 4,  R2 = 16; };
template <> struct XPlan<4096>  { static constexpr int R1 = 8,  R2 = 16; };
template <> struct XPlan<8192>  { static constexpr int R1 = 16, R2 = 16; };
template <> struct XPlan<16384> { static constexpr int R1 = 32, R2 = 16; };

// 32nd roots of unity e^{+2 pi i j/32} (exact to fp32 rounding): the integer part b of the shift
// is the rotation e^{i theta_k b}; for the 16 modes k = klow + (N/32) q of one thread it is
// base * root32[(b q) mod 32]; the 32 roots travel in the kernel argument block (constant bank).

__device__ __forceinline__ int swz(int c) { return c ^ ((c >> 3) & 7); }

__device__ __forceinline__ void cp_async16(void* smem, const void* gmem)
{
    const unsigned s = (unsigned)__cvta_generic_to_shared(smem);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(s), "l"(gmem) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;\n" ::: "memory"); }

// Un-rotated symbol at (c, s) = (cos theta, sin theta): Lagrange 2d+1 in Everett form
//   P(sv; 1-b*) + e^{i theta} P(sv; b*),  sv = 2 - 2c,  P(sv;t) = sum_k a_k(t) sv^k
// cubic spline: [B(b*+1) e^{-i theta} + B(b*) + B(b*-1) e^{i theta} + B(b*-2) e^{2 i theta}] 3/(2+c).
// The coefficient arrays carry the 1/(2N) of the real-FFT halves and the inverse normalisation.
template <int SYM> struct SymCoef {
    static constexpr int D = SYM == SYM_LAG_D1 ? 1 : (SYM == SYM_LAG_D4 ? 4 : (SYM == SYM_LAG_D8 ? 8 : 3));
    float a1[D + 1], a2[D + 1];   // spline: a1[0..3] = Bm1, B0, B1, B2
};

template <int SYM>
__device__ __forceinline__ void sym_load(SymCoef<SYM>& k, const float* __restrict__ rec)
{
    if constexpr (SYM == SYM_SPLINE3) {
#pragma unroll
        for (int i = 0; i < 4; ++i) k.a1[i] = rec[4 + i];
    } else {
#pragma unroll
        for (int i = 0; i <= SymCoef<SYM>::D; ++i) { k.a1[i] = rec[4 + i]; k.a2[i] = rec[13 + i]; }
    }
}

template <int SYM>
__device__ __forceinline__ float2 sym_eval(const SymCoef<SYM>& k, const float c, const float s)
{
    if constexpr (SYM == SYM_SPLINE3) {
        const float Bm1 = k.a1[0], B0 = k.a1[1], B1 = k.a1[2], B2 = k.a1[3];
        const float c2 = fmaf(2.0f * c, c, -1.0f), s2 = 2.0f * s * c;
        const float g = __fdividef(1.0f, 2.0f + c);
        const float lr = fmaf(B2, c2, fmaf(Bm1 + B1, c, B0)) * g;
        const float li = fmaf(B2, s2, (B1 - Bm1) * s) * g;
        return make_float2(lr, li);
    } else {
        constexpr int D = SymCoef<SYM>::D;
        const float sv = fmaf(-2.0f, c, 2.0f);
        float p1 = k.a1[D], p2 = k.a2[D];
#pragma unroll
        for (int i = D - 1; i >= 0; --i) { p1 = fmaf(p1, sv, k.a1[i]); p2 = fmaf(p2, sv, k.a2[i]); }
        return make_float2(fmaf(c, p2, p1), s * p2);
    }
}


// ---------------------------------------------------------------------------------------------
// shared-memory accessors: the buffer is an array of 16-byte chunks (2 complex), physical chunk
// index = swz(logical chunk index)
__device__ __forceinline__ float4 lds4(const float4* b, int pc) { return b[pc]; }

// strided pass, two adjacent positions per thread (VEC = 2): logical chunks c0 + k*SC
template <int R, int SC>
struct PairAddr {
    int base;
    __device__ __forceinline__ explicit PairAddr(int c0)
    {
        if constexpr (SC % 64 == 0) base = c0 ^ ((c0 >> 3) & 7); else base = c0;
    }
    __device__ __forceinline__ int at(int k) const
    {
        if constexpr (SC % 64 == 0) return base + k * SC; else return swz(base + k * SC);
    }
};

template <int R, int S1>
__device__ __forceinline__ void fwd_pair_pass(float4* __restrict__ buf, const int c0, const int tp,
                                              const float2* __restrict__ tw)
{
    constexpr int SC = S1 / 2;
    const PairAddr<R, SC> A(c0);
    float2 x0[R], x1[R];
#pragma unroll
    for (int k = 0; k < R; ++k) {
        const float4 v = buf[A.at(k)];
        x0[k] = make_float2(v.x, v.y);
        x1[k] = make_float2(v.z, v.w);
    }
    dft_dif<R, 1>(x0);
    dft_dif<R, 1>(x1);
    buf[A.at(0)] = make_float4(x0[0].x, x0[0].y, x1[0].x, x1[0].y);
    const float4* __restrict__ tw4 = reinterpret_cast<const float4*>(tw) + tp;
#pragma unroll
    for (int q = 1; q < R; ++q) {
        const float4 w = __ldg(tw4 + (q - 1) * SC);
        const float2 y0 = cmul(x0[brev(q, R)], make_float2(w.x, w.y));
        const float2 y1 = cmul(x1[brev(q, R)], make_float2(w.z, w.w));
        buf[A.at(q)] = make_float4(y0.x, y0.y, y1.x, y1.y);
    }
}

// inverse of fwd_pair_pass; if GOUT the natural-order result goes to global memory (gout = the
// line as float4, chunk index = logical chunk), else back to shared memory.
template <int R, int S1, bool GOUT>
__device__ __forceinline__ void inv_pair_pass(float4* __restrict__ buf, const int c0, const int tp,
                                              const float2* __restrict__ tw, float4* __restrict__ gout,
                                              const float dc)
{
    constexpr int SC = S1 / 2;
    const PairAddr<R, SC> A(c0);
    float2 x0[R], x1[R];
    {
        const float4 v = buf[A.at(0)];
        x0[0] = make_float2(v.x, v.y);
        x1[0] = make_float2(v.z, v.w);
    }
    const float4* __restrict__ tw4 = reinterpret_cast<const float4*>(tw) + tp;
#pragma unroll
    for (int q = 1; q < R; ++q) {
        const float4 v = buf[A.at(q)];
        const float4 w = __ldg(tw4 + (q - 1) * SC);
        x0[brev(q, R)] = cmulc(make_float2(v.x, v.y), make_float2(w.x, w.y));
        x1[brev(q, R)] = cmulc(make_float2(v.z, v.w), make_float2(w.z, w.w));
    }
    idft_dit<R, 1>(x0);
    idft_dit<R, 1>(x1);
#pragma unroll
    for (int k = 0; k < R; ++k) {
        if constexpr (GOUT)
            __stcs(gout + tp + k * SC, make_float4(x0[k].x + dc, x0[k].y + dc, x1[k].x + dc, x1[k].y + dc));
        else buf[A.at(k)] = make_float4(x0[k].x, x0[k].y, x1[k].x, x1[k].y);
    }
}

// strided pass, one position per thread (VEC = 1; used for radix 32): logical elements e0 + k*S1
template <int S1>
__device__ __forceinline__ int elem_addr(const int e)   // float2 index of logical element e
{
    return (swz(e >> 1) << 1) | (e & 1);
}

template <int R, int S1>
__device__ __forceinline__ void fwd_single_pass(float2* __restrict__ buf, const int e0, const int t,
                                                const float2* __restrict__ tw)
{
    float2 x[R];
    int a0;
    if constexpr (S1 % 128 == 0) a0 = elem_addr<S1>(e0);
#pragma unroll
    for (int k = 0; k < R; ++k) x[k] = buf[(S1 % 128 == 0) ? a0 + k * S1 : elem_addr<S1>(e0 + k * S1)];
    dft_dif<R, 1>(x);
    buf[(S1 % 128 == 0) ? a0 : elem_addr<S1>(e0)] = x[0];
#pragma unroll
    for (int q = 1; q < R; ++q)
        buf[(S1 % 128 == 0) ? a0 + q * S1 : elem_addr<S1>(e0 + q * S1)] = cmul(x[brev(q, R)], __ldg(tw + (q - 1) * S1 + t));
}

template <int R, int S1, bool GOUT>
__device__ __forceinline__ void inv_single_pass(float2* __restrict__ buf, const int e0, const int t,
                                                const float2* __restrict__ tw, float2* __restrict__ gout,
                                                const float dc)
{
    float2 x[R];
    int a0;
    if constexpr (S1 % 128 == 0) a0 = elem_addr<S1>(e0);
    x[0] = buf[(S1 % 128 == 0) ? a0 : elem_addr<S1>(e0)];
#pragma unroll
    for (int q = 1; q < R; ++q)
        x[brev(q, R)] = cmulc(buf[(S1 % 128 == 0) ? a0 + q * S1 : elem_addr<S1>(e0 + q * S1)], __ldg(tw + (q - 1) * S1 + t));
    idft_dit<R, 1>(x);
#pragma unroll
    for (int k = 0; k < R; ++k) {
        if constexpr (GOUT) __stcs(gout + t + k * S1, make_float2(x[k].x + dc, x[k].y + dc));
        else buf[(S1 % 128 == 0) ? a0 + k * S1 : elem_addr<S1>(e0 + k * S1)] = x[k];
    }
}

// middle pass (three-pass sizes): radix 16, stride 16 complex inside sub-blocks of 256 complex
// (128 chunks); cb = logical chunk of the sub-block start (a multiple of 64), tp in [0, 8).
template <bool INV>
__device__ __forceinline__ void mid_pass(float4* __restrict__ buf, const int cb, const int tp,
                                         const float2* __restrict__ tw)
{
    float2 x0[16], x1[16];
    int off[8];
#pragma unroll
    for (int k = 0; k < 8; ++k) off[k] = cb + 8 * k + (tp ^ k);
    const float4* __restrict__ tw4 = reinterpret_cast<const float4*>(tw) + tp;
    if constexpr (!INV) {
#pragma unroll
        for (int k = 0; k < 16; ++k) {
            const float4 v = buf[off[k & 7] + (k & 8) * 8];
            x0[k] = make_float2(v.x, v.y);
            x1[k] = make_float2(v.z, v.w);
        }
        dft_dif<16, 1>(x0);
        dft_dif<16, 1>(x1);
        buf[off[0]] = make_float4(x0[0].x, x0[0].y, x1[0].x, x1[0].y);
#pragma unroll
        for (int q = 1; q < 16; ++q) {
            const float4 w = __ldg(tw4 + (q - 1) * 8);
            const float2 y0 = cmul(x0[brev(q, 16)], make_float2(w.x, w.y));
            const float2 y1 = cmul(x1[brev(q, 16)], make_float2(w.z, w.w));
            buf[off[q & 7] + (q & 8) * 8] = make_float4(y0.x, y0.y, y1.x, y1.y);
        }
    } else {
        {
            const float4 v = buf[off[0]];
            x0[0] = make_float2(v.x, v.y);
            x1[0] = make_float2(v.z, v.w);
        }
#pragma unroll
        for (int q = 1; q < 16; ++q) {
            const float4 v = buf[off[q & 7] + (q & 8) * 8];
            const float4 w = __ldg(tw4 + (q - 1) * 8);
            x0[brev(q, 16)] = cmulc(make_float2(v.x, v.y), make_float2(w.x, w.y));
            x1[brev(q, 16)] = cmulc(make_float2(v.z, v.w), make_float2(w.z, w.w));
        }
        idft_dit<16, 1>(x0);
        idft_dit<16, 1>(x1);
#pragma unroll
        for (int k = 0; k < 16; ++k)
            buf[off[k & 7] + (k & 8) * 8] = make_float4(x0[k].x, x0[k].y, x1[k].x, x1[k].y);
    }
}


// ---------------------------------------------------------------------------------------------
// One mirror pair (k, M-k) of the half-length spectrum: untangle, symbol, re-tangle.
//   P = Z_k, Qm = Z_{M-k};  cs = (cos, sin)(2 pi k / N);  rot = e^{i theta_k b};  sgn = (-1)^b.
template <int SYM>
__device__ __forceinline__ void pair_op(float2& P, float2& Qm, const float2 cs, const float2 rot,
                                        const float sgn, const SymCoef<SYM>& K)
{
    const float c = cs.x, s = cs.y;
    const float2 E2 = make_float2(P.x + Qm.x, P.y - Qm.y);      // P + conj(Qm)
    const float2 D2 = make_float2(P.x - Qm.x, P.y + Qm.y);      // P - conj(Qm)
    // T2 = W_N^k (-i D2),  W_N^k = (c, -s)
    const float2 T2 = make_float2(fmaf(c, D2.y, -s * D2.x), -fmaf(c, D2.x, s * D2.y));
    const float2 Up = cadd(E2, T2), Um = csub(E2, T2);           // 2 U_k, 2 conj(U_{M-k})
    const float2 la = sym_eval<SYM>(K, c, s);
    const float2 lm = sym_eval<SYM>(K, -c, s);                   // theta_{M-k} = pi - theta_k
    const float2 a = cmul(rot, la);                              // lambda_k / (2N)
    const float2 cc = cmul(rot, make_float2(sgn * lm.x, -sgn * lm.y));   // conj(lambda_{M-k}) / (2N)
    const float2 Vp = cmul(a, Up), Vm = cmul(cc, Um);
    const float2 Ep = cadd(Vp, Vm), Dp = csub(Vp, Vm);
    const float2 Op = make_float2(fmaf(c, Dp.x, -s * Dp.y), fmaf(c, Dp.y, s * Dp.x));   // conj(W) Dp
    P = make_float2(Ep.x - Op.y, Ep.y + Op.x);                   // E' + i O'
    Qm = make_float2(Ep.x + Op.y, Op.x - Ep.y);                  // conj(E' - i O')
}

// e^{+2 pi i j / N} from the half-circle table cs[k] = (cos, sin)(2 pi k/N), k = 0..N/2
template <int N>
__device__ __forceinline__ float2 unit_root(const float2* __restrict__ cs, int j)
{
    j &= N - 1;
    const bool up = j > N / 2;
    const float2 v = __ldg(cs + (up ? N - j : j));
    return make_float2(v.x, up ? -v.y : v.y);
}

// Fused middle stage on one item = two radix-16 groups gA, gB whose modes mirror each other:
// pair slot q holds (Z_k, Z_{M-k}) in (XA[brev q], XB[brev(15-q)]), k = klowA + ML q.
// The one "special" item per line (gA = group 0, gB = the self-mirrored group) is brought to the
// same form by a register permutation (executed by that thread's warp only):
//   slots 0..7  : group B pairs  (q, 15-q),      k = ML/2 + ML q
//   slots 8..14 : group A pairs  (q', 16-q'),    k = ML q',  q' = slot - 7
//   slot  15    : k = M/2, its own mirror;   k = 0 (with k = M, the line's Nyquist mode) apart.
template <int N, int SYM>
__device__ __forceinline__ void symbol_item_x(float4* __restrict__ buf, const int cline, const int gA,
                                              const int gB, const int klowA, const bool special,
                                              float* __restrict__ rec, const float2* __restrict__ cs,
                                              const float2* ROOT32)
{
    constexpr int M = N / 2, ML = M / 16;
    float2 XA[16], XB[16];
    const int pa = cline + gA * 8, pb = cline + gB * 8;
    const int xa = (pa >> 3) & 7, xb = (pb >> 3) & 7;
#pragma unroll
    for (int j = 0; j < 8; ++j) {
        const float4 va = buf[pa + (j ^ xa)], vb = buf[pb + (j ^ xb)];
        XA[2 * j] = make_float2(va.x, va.y); XA[2 * j + 1] = make_float2(va.z, va.w);
        XB[2 * j] = make_float2(vb.x, vb.y); XB[2 * j + 1] = make_float2(vb.z, vb.w);
    }
    dft_dif<16, 1>(XA);
    dft_dif<16, 1>(XB);
    float2 z0 = XA[0];
    if (special) {
        float2 TA[16];
#pragma unroll
        for (int i = 0; i < 16; ++i) TA[i] = XA[i];
#pragma unroll
        for (int q = 0; q < 8; ++q) XA[brev(q, 16)] = XB[brev(q, 16)];
#pragma unroll
        for (int q = 8; q < 15; ++q) { XA[brev(q, 16)] = TA[brev(q - 7, 16)]; XB[brev(15 - q, 16)] = TA[brev(23 - q, 16)]; }
        XA[brev(15, 16)] = TA[brev(8, 16)];
        XB[brev(0, 16)] = TA[brev(8, 16)];
    }
    SymCoef<SYM> K;
    sym_load<SYM>(K, rec);
    const int b = __float_as_int(rec[0]);
    const float sgn = (b & 1) ? -1.0f : 1.0f;
    const int klo = special ? ML / 2 : klowA;            // slots 0..7
    const int khi = special ? ML / 2 - 15 * ML / 2 : klowA;   // slots 8..15: k = khi + ML q
    const float2 base_lo = unit_root<N>(cs, b * klo);
    const float2 base_hi = unit_root<N>(cs, b * khi);
#pragma unroll
    for (int q = 0; q < 16; ++q) {
        const float2 rot = cmul(q < 8 ? base_lo : base_hi, ROOT32[(b * q) & 31]);
        pair_op<SYM>(XA[brev(q, 16)], XB[brev(15 - q, 16)], __ldg(cs + (q < 8 ? klo : khi) + ML * q), rot, sgn, K);
    }
    if (special) {
        // back to group order: XA[brev i] = Z'_{ML i}, XB[brev i] = Z'_{ML/2 + ML i}
        float2 TA[16], TB[8];
#pragma unroll
        for (int i = 0; i < 16; ++i) TA[i] = XA[i];
#pragma unroll
        for (int j = 1; j < 8; ++j) TB[j] = XB[brev(j, 16)];                  // Q'_{15-j} = Z'_{ML (8+j)}
#pragma unroll
        for (int q = 0; q < 8; ++q) XB[brev(q, 16)] = TA[brev(q, 16)];        // P'_q = Z'_{ML/2 + ML q}
#pragma unroll
        for (int i = 1; i < 8; ++i) {
            XA[brev(i, 16)] = TA[brev(i + 7, 16)];                            // P'_{i+7} = Z'_{ML i}
            XA[brev(16 - i, 16)] = TB[8 - i];                                 // Q'_{i+7} = Z'_{ML (16-i)}
        }
        XA[brev(8, 16)] = TA[brev(15, 16)];                                   // P'_15 = Z'_{M/2}
        // k = 0 and k = M: U_0 = x + y, U_M = x - y, lambda_0 = 1 exactly.  The line mean A0 by-passes
        // the inverse transform (added back in the last pass): the intermediate sums then stay at
        // fluctuation level, with one rounding at the level of the mean.
        const float A0 = rec[1] * (z0.x + z0.y), Bn = rec[2] * (z0.x - z0.y);
        XA[0] = make_float2(Bn, -Bn);
        rec[3] = A0;
    }
    idft_dit<16, 1>(XA);
    idft_dit<16, 1>(XB);
#pragma unroll
    for (int j = 0; j < 8; ++j) {
        buf[pa + (j ^ xa)] = make_float4(XA[2 * j].x, XA[2 * j].y, XA[2 * j + 1].x, XA[2 * j + 1].y);
        buf[pb + (j ^ xb)] = make_float4(XB[2 * j].x, XB[2 * j].y, XB[2 * j + 1].x, XB[2 * j + 1].y);
    }
}

// mirror-pair enumeration of the radix-16 groups of one line: item u in [0, M/32)
template <int R1, int R2>
__device__ __forceinline__ void item_groups(const int u, int& gA, int& gB, int& klowA, bool& special)
{
    if constexpr (R2 == 1) {
        special = (u == 0);
        gA = u; klowA = u;
        gB = special ? R1 / 2 : R1 - u;
    } else {
        const int row = u / R2, r = u & (R2 - 1);
        int q1, q2;
        if (row < R1 / 2 - 1) { q1 = row + 1; q2 = r; }
        else if (r < R2 / 2)  { q1 = 0; q2 = r; }
        else                  { q1 = R1 / 2; q2 = r - R2 / 2; }
        special = (q1 == 0 && q2 == 0);
        gA = q1 * R2 + q2;
        klowA = q1 + R1 * q2;
        const int q1b = (R1 - q1) & (R1 - 1);
        const int q2b = special ? R2 / 2 : (q1 ? R2 - 1 - q2 : R2 - q2);
        gB = q1b * R2 + q2b;
    }
}


template <int N, int SYM>
__global__ void __launch_bounds__(128, 4) advect_x_kernel(const AdvectXArgs a)
{
    using PL = XPlan<N>;
    constexpr int M = N / 2, R1 = PL::R1, R2 = PL::R2;
    constexpr int S1 = M / R1;
    constexpr bool PAIR_A = (R1 <= 16);
    constexpr int ITEMS_A = PAIR_A ? S1 / 2 : S1;
    constexpr int ITEMS_C = M / 32;
    constexpr int CH = M / 2;                     // 16-byte chunks per line
    constexpr int RCH = XREC_WORDS / 4;           // 16-byte chunks per record

    extern __shared__ __align__(1024) unsigned char smem_raw[];
    const int lpi = 1 << a.lpi_log;
    const int nbuf = a.nbuf;                                                      // 1 or 2 line buffers
    float4* const bufs = reinterpret_cast<float4*>(smem_raw);                     // nbuf x lpi x CH chunks
    float4* const recs4 = bufs + nbuf * lpi * CH;                                 // nbuf x lpi x RCH chunks
    const int tid = threadIdx.x, T = blockDim.x;

    auto prefetch = [&](int g, int sel) {
        float4* dst = bufs + sel * lpi * CH;
        const float4* src = reinterpret_cast<const float4*>(a.f) + (size_t)g * lpi * CH;
        for (int i = tid; i < lpi * CH; i += T) cp_async16(dst + swz(i), src + i);
        float4* rdst = recs4 + sel * lpi * RCH;
        const float4* rsrc = reinterpret_cast<const float4*>(a.rec) + (size_t)g * lpi * RCH;
        for (int i = tid; i < lpi * RCH; i += T) cp_async16(rdst + i, rsrc + i);
    };

    pdl_wait();                                   // shift records and grid come from the kernels before
    pdl_launch_dependents();
    int g = blockIdx.x;
    if (g < a.n_groups) prefetch(g, 0);
    cp_async_commit();
    for (int it = 0; g < a.n_groups; g += gridDim.x, ++it) {
        const int sel = nbuf == 2 ? (it & 1) : 0;
        if (nbuf == 1 && it > 0) {                 // single buffer: reload after everybody left iteration it-1
            __syncthreads();
            prefetch(g, 0);
            cp_async_commit();
        }
        cp_async_wait_all();
        __syncthreads();                           // group g landed; everybody left iteration it-1
        if (nbuf == 2) {
            if (g + (int)gridDim.x < a.n_groups) prefetch(g + gridDim.x, sel ^ 1);
            cp_async_commit();
        }
        float4* const buf = bufs + sel * lpi * CH;
        float* const recs = reinterpret_cast<float*>(recs4 + sel * lpi * RCH);

        // ---- forward pass A
#pragma unroll 1
        for (int w = tid; w < lpi * ITEMS_A; w += T) {
            const int l = w / ITEMS_A, t = w & (ITEMS_A - 1);
            if constexpr (PAIR_A) fwd_pair_pass<R1, S1>(buf, l * CH + t, t, a.twA);
            else fwd_single_pass<R1, S1>(reinterpret_cast<float2*>(buf), l * M + t, t, a.twA);
        }
        __syncthreads();
        // ---- forward pass B
        if constexpr (R2 == 16) {
#pragma unroll 1
            for (int w = tid; w < lpi * ITEMS_C; w += T) {
                const int l = w / ITEMS_C, i = w & (ITEMS_C - 1);
                mid_pass<false>(buf, l * CH + (i >> 3) * 128, i & 7, a.twB);
            }
            __syncthreads();
        }
        // ---- symbol stage
#pragma unroll 1
        for (int w = tid; w < lpi * ITEMS_C; w += T) {
            const int l = w / ITEMS_C, u = w & (ITEMS_C - 1);
            int gA, gB, klowA;
            bool special;
            item_groups<R1, R2>(u, gA, gB, klowA, special);
            float* rec = recs + l * XREC_WORDS;
            symbol_item_x<N, SYM>(buf, l * CH, gA, gB, klowA, special, rec, a.cs, a.root32);
        }
        __syncthreads();
        // ---- inverse pass B
        if constexpr (R2 == 16) {
#pragma unroll 1
            for (int w = tid; w < lpi * ITEMS_C; w += T) {
                const int l = w / ITEMS_C, i = w & (ITEMS_C - 1);
                mid_pass<true>(buf, l * CH + (i >> 3) * 128, i & 7, a.twB);
            }
            __syncthreads();
        }
        // ---- inverse pass A: shared -> registers -> global
        float4* const gout = reinterpret_cast<float4*>(a.f) + (size_t)g * lpi * CH;
#pragma unroll 1
        for (int w = tid; w < lpi * ITEMS_A; w += T) {
            const int l = w / ITEMS_A, t = w & (ITEMS_A - 1);
            const float dc = recs[l * XREC_WORDS + 3];
            if constexpr (PAIR_A) inv_pair_pass<R1, S1, true>(buf, l * CH + t, t, a.twA, gout + l * CH, dc);
            else inv_single_pass<R1, S1, true>(reinterpret_cast<float2*>(buf), l * M + t, t, a.twA,
                                               reinterpret_cast<float2*>(gout + l * CH), dc);
        }
    }
}

}  // namespace vog
