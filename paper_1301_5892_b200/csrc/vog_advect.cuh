// vog_advect.cuh -- the fused per-line advection kernel.
//
// One CTA owns NL complex lines (= 2*NL real lines: velocity rows for the x-direction, space
// columns for the v-direction).  Each line goes global -> registers -> shared memory through
// the first radix pass, stays in shared memory for the remaining forward passes, meets its
// symbol lambda_m (the eigenvalues D = FFT(a) of the circulant A, evaluated in
// closed form instead of transforming a) in registers between the last forward and the first
// inverse pass, and leaves through the last inverse pass straight to global memory.  The
// phase-space array is read once and written once per advection.
//
// x-direction (VDIR=false): a complex line is rows (r, r+1); lanes run along x (coalesced).
// v-direction (VDIR=true): a complex line is columns (i, i+1), loaded as one float2 per row;
//   lanes run across the NL lines of the tile first (2*NL adjacent columns = 8*NL bytes per
//   row), the "transposed tile": no transposition pass exists (contrast P:157, 169-171).
#pragma once
#include "vog_fft.cuh"
#include "vog_internal.h"

namespace vog {

template <int SYM> struct SymDeg { static constexpr int D = SYM == SYM_LAG_D1 ? 1 : (SYM == SYM_LAG_D4 ? 4 : 8); };

// V[q] *= lambda_{m(q)} for the 16 modes of a symbol-stage item, one real line (record rec).
// Lagrange 2d+1, Everett form: lambda = e^{i theta b} [P(s;1-b*) + e^{i theta} P(s;b*)],
//   s = 2 - 2 cos(theta), P(s;t) = sum_k a_k(t) s^k, a_k(t) = (-1)^k C(t+k, 2k+1) >= 0.
// Cubic spline: lambda = e^{i theta b} [B(b*+1)e^{-i theta} + B(b*) + B(b*-1)e^{i theta}
//   + B(b*-2)e^{2 i theta}] * 3/(2 + cos(theta)).
// The records carry the 1/(2N) (two-for-one split and inverse-FFT normalisation).
template <int N, int SYM, typename ModeFn>
__device__ __forceinline__ void apply_symbol(float2 (&V)[16], const float* __restrict__ rec,
                                             const float2* __restrict__ tw, ModeFn mode)
{
    const int b = __float_as_int(rec[0]);
    if constexpr (SYM == SYM_SPLINE3) {
        const float Bm1 = rec[1], B0 = rec[2], B1 = rec[3], B2 = rec[4];
        const float Bs = Bm1 + B1, Bd = B1 - Bm1;
#pragma unroll
        for (int q = 0; q < 16; ++q) {
            const int m = mode(q);
            const float2 t1 = __ldg(tw + m);
            const float c = t1.x, s = -t1.y;
            const float c2 = fmaf(2.0f * c, c, -1.0f), s2 = 2.0f * s * c;
            const float g = __fdividef(1.0f, 2.0f + c);
            const float lr = fmaf(B2, c2, fmaf(Bs, c, B0)) * g;
            const float li = fmaf(B2, s2, Bd * s) * g;
            const float2 r = __ldg(tw + ((m * b) & (N - 1)));
            const float2 lam = cmulc(make_float2(lr, li), r);
            V[q] = cmul(lam, V[q]);
        }
    } else {
        constexpr int D = SymDeg<SYM>::D;
        float a1[D + 1], a2[D + 1];
#pragma unroll
        for (int k = 0; k <= D; ++k) { a1[k] = rec[1 + k]; a2[k] = rec[10 + k]; }
#pragma unroll
        for (int q = 0; q < 16; ++q) {
            const int m = mode(q);
            const float2 t1 = __ldg(tw + m);
            const float c = t1.x, s = -t1.y;
            const float sv = fmaf(-2.0f, c, 2.0f);
            float p1 = a1[D], p2 = a2[D];
#pragma unroll
            for (int k = D - 1; k >= 0; --k) { p1 = fmaf(p1, sv, a1[k]); p2 = fmaf(p2, sv, a2[k]); }
            const float lr = fmaf(c, p2, p1), li = s * p2;
            const float2 r = __ldg(tw + ((m * b) & (N - 1)));
            const float2 lam = cmulc(make_float2(lr, li), r);
            V[q] = cmul(lam, V[q]);
        }
    }
}

// Symbol-stage item: last forward radix-16 pass on two groups (A, B) whose modes are mutual
// mirrors m <-> N-m, two-for-one separation, symbol multiply for both real lines, recombination,
// first inverse radix-16 pass.  SPECIAL = the item holding the self-mirrored modes 0 and N/2
// (groups m_low = 0 and m_low = N/32).
template <int N, int SYM, bool SPECIAL>
__device__ __forceinline__ void symbol_item(float2* __restrict__ smc, const int SP, const int gA, const int gB,
                                            const int mlowA, const float* __restrict__ recA,
                                            const float* __restrict__ recB, const float2* __restrict__ tw)
{
    constexpr int ML = N / 16;
    float2 XA[16], XB[16];
#pragma unroll
    for (int k = 0; k < 16; ++k) {
        XA[k] = smc[padp(gA * 16 + k) * SP];
        XB[k] = smc[padp(gB * 16 + k) * SP];
    }
    dft_dif<16, 1>(XA);
    dft_dif<16, 1>(XB);
    // pair slots: (Pv[q], Qv[q]) = (Z_m, Z_{N-m}), m = mode(q)
    float2 Pv[16], Qv[16];
    if constexpr (!SPECIAL) {
#pragma unroll
        for (int q = 0; q < 16; ++q) { Pv[q] = XA[brev(q, 16)]; Qv[q] = XB[brev(15 - q, 16)]; }
    } else {
#pragma unroll
        for (int q = 0; q < 8; ++q) { Pv[q] = XB[brev(q, 16)]; Qv[q] = XB[brev(15 - q, 16)]; }
#pragma unroll
        for (int q = 1; q < 8; ++q) { Pv[7 + q] = XA[brev(q, 16)]; Qv[7 + q] = XA[brev(16 - q, 16)]; }
        Pv[15] = XA[brev(8, 16)]; Qv[15] = XA[brev(8, 16)];   // Nyquist, self-mirrored
    }
    auto mode = [&](int q) -> int {
        if constexpr (!SPECIAL) return mlowA + ML * q;
        else return q < 8 ? ML / 2 + ML * q : (q < 15 ? ML * (q - 7) : N / 2);
    };
    // U_A = (Z_m + conj Z_{N-m})/2, U_B = (Z_m - conj Z_{N-m})/(2i); the 1/2 lives in the records
#pragma unroll
    for (int q = 0; q < 16; ++q) {
        const float2 p = Pv[q], z = Qv[q];
        Pv[q] = make_float2(p.x + z.x, p.y - z.y);
        Qv[q] = make_float2(p.y + z.y, z.x - p.x);
    }
    apply_symbol<N, SYM>(Pv, recA, tw, mode);
    apply_symbol<N, SYM>(Qv, recB, tw, mode);
    // Y_m = W_A + i W_B,  Y_{N-m} = conj(W_A) + i conj(W_B)
#pragma unroll
    for (int q = 0; q < 16; ++q) {
        const float2 wa = Pv[q], wb = Qv[q];
        Pv[q] = make_float2(wa.x - wb.y, wa.y + wb.x);
        Qv[q] = make_float2(wa.x + wb.y, wb.x - wa.y);
    }
    if constexpr (!SPECIAL) {
#pragma unroll
        for (int q = 0; q < 16; ++q) { XA[brev(q, 16)] = Pv[q]; XB[brev(15 - q, 16)] = Qv[q]; }
    } else {
#pragma unroll
        for (int q = 0; q < 8; ++q) { XB[brev(q, 16)] = Pv[q]; XB[brev(15 - q, 16)] = Qv[q]; }
#pragma unroll
        for (int q = 1; q < 8; ++q) { XA[brev(q, 16)] = Pv[7 + q]; XA[brev(16 - q, 16)] = Qv[7 + q]; }
        XA[brev(8, 16)] = Pv[15];
        // mode 0: lambda_0 = sum of the interpolation weights = 1 exactly; only the 1/N remains
        XA[0].x *= 1.0f / (float)N;
        XA[0].y *= 1.0f / (float)N;
    }
    idft_dit<16, 1>(XA);
    idft_dit<16, 1>(XB);
#pragma unroll
    for (int k = 0; k < 16; ++k) {
        smc[padp(gA * 16 + k) * SP] = XA[k];
        smc[padp(gB * 16 + k) * SP] = XB[k];
    }
}

// forward pass, shared -> shared: sub-blocks of length B, radix R, stride S = B/R
template <int N, int R, int B>
__device__ __forceinline__ void fwd_pass_smem(float2* __restrict__ smc, const int SP, const int g,
                                              const float2* __restrict__ tw)
{
    constexpr int S = B / R;
    const int t = g & (S - 1);
    const int base = (g / S) * B + t;
    float2 x[R];
#pragma unroll
    for (int k = 0; k < R; ++k) x[k] = smc[padp(base + k * S) * SP];
    dft_dif<R, 1>(x);
    smc[padp(base) * SP] = x[0];
    const int tm = t * (N / B);
#pragma unroll
    for (int q = 1; q < R; ++q)
        smc[padp(base + q * S) * SP] = cmul(x[brev(q, R)], __ldg(tw + tm * q));
}

template <int N, int R, int B>
__device__ __forceinline__ void inv_pass_smem(float2* __restrict__ smc, const int SP, const int g,
                                              const float2* __restrict__ tw)
{
    constexpr int S = B / R;
    const int t = g & (S - 1);
    const int base = (g / S) * B + t;
    const int tm = t * (N / B);
    float2 x[R];
    x[0] = smc[padp(base) * SP];
#pragma unroll
    for (int q = 1; q < R; ++q)
        x[brev(q, R)] = cmulc(smc[padp(base + q * S) * SP], __ldg(tw + tm * q));
    idft_dit<R, 1>(x);
#pragma unroll
    for (int k = 0; k < R; ++k) smc[padp(base + k * S) * SP] = x[k];
}

template <int N, int SYM, bool VDIR>
__global__ void __launch_bounds__(512) advect_kernel(const AdvectArgs a)
{
    using RX = Radix<N>;
    constexpr int R1 = RX::R1, R2 = RX::R2, P = RX::P;
    constexpr int S1 = N / R1;           // butterflies per line in pass 1
    constexpr int ML = N / 16;           // radix-16 groups per line
    constexpr int IT = ML / 2;           // symbol-stage items per line
    constexpr int PL = padded_len(N);

    extern __shared__ __align__(16) unsigned char smem_raw[];
    float2* sm = reinterpret_cast<float2*>(smem_raw);
    const int lognl = a.lognl;
    const int NL = 1 << lognl;
    float* recs = reinterpret_cast<float*>(sm + (size_t)NL * PL);

    const int tid = threadIdx.x, T = blockDim.x;
    const int line0 = blockIdx.x * 2 * NL;          // first real line (row or column) of this tile
    const int SP = VDIR ? NL : 1;
    const int SC = VDIR ? 1 : PL;
    const int Nx = a.Nx;
    const float2* __restrict__ tw = a.tw;

    pdl_wait();                                   // shift records and grid come from the kernels before
    pdl_launch_dependents();
    for (int i = tid; i < 2 * NL * REC_WORDS; i += T) recs[i] = a.rec[(size_t)line0 * REC_WORDS + i];

    // ---- forward pass 1: global -> registers -> shared
    for (int w = tid; w < NL * S1; w += T) {
        int c, t;
        if (VDIR) { c = w & (NL - 1); t = w >> lognl; } else { c = w / S1; t = w & (S1 - 1); }
        float2 x[R1];
        if (VDIR) {
#pragma unroll
            for (int k = 0; k < R1; ++k)
                x[k] = __ldcs(reinterpret_cast<const float2*>(a.f + (size_t)(t + k * S1) * Nx + line0 + 2 * c));
        } else {
            const float* fa = a.f + (size_t)(line0 + 2 * c) * Nx + t;
#pragma unroll
            for (int k = 0; k < R1; ++k) { x[k].x = __ldcs(fa + k * S1); x[k].y = __ldcs(fa + Nx + k * S1); }
        }
        dft_dif<R1, 1>(x);
        float2* smc = sm + c * SC;
        smc[padp(t) * SP] = x[0];
#pragma unroll
        for (int q = 1; q < R1; ++q)
            smc[padp(t + q * S1) * SP] = cmul(x[brev(q, R1)], __ldg(tw + t * q));
    }
    __syncthreads();

    // ---- forward pass 2 (three-pass sizes)
    if constexpr (P == 3) {
        constexpr int G2 = N / R2;
        for (int w = tid; w < NL * G2; w += T) {
            int c, g;
            if (VDIR) { c = w & (NL - 1); g = w >> lognl; } else { c = w / G2; g = w & (G2 - 1); }
            fwd_pass_smem<N, R2, N / R1>(sm + c * SC, SP, g, tw);
        }
        __syncthreads();
    }

    // ---- symbol stage: last forward pass + lambda + first inverse pass, in registers
    for (int w = tid; w < NL * IT; w += T) {
        int c, u;
        if (VDIR) { c = w & (NL - 1); u = w >> lognl; } else { c = w / IT; u = w & (IT - 1); }
        int gA, gB, mlowA;
        bool special;
        if constexpr (P == 2) {
            special = (u == 0);
            gA = u; mlowA = u;
            gB = special ? R1 / 2 : R1 - u;
        } else {
            const int row = u / R2, r = u & (R2 - 1);
            int q1, q2;
            if (row < R1 / 2 - 1) { q1 = row + 1; q2 = r; }
            else if (r < R2 / 2)  { q1 = 0; q2 = r; }
            else                  { q1 = R1 / 2; q2 = r - R2 / 2; }
            special = (q1 == 0 && q2 == 0);
            gA = q1 * R2 + q2;
            mlowA = q1 + R1 * q2;
            const int q1b = (R1 - q1) & (R1 - 1);
            const int q2b = special ? R2 / 2 : (q1 ? R2 - 1 - q2 : R2 - q2);
            gB = q1b * R2 + q2b;
        }
        const float* recA = recs + (2 * c) * REC_WORDS;
        const float* recB = recA + REC_WORDS;
        if (special) symbol_item<N, SYM, true>(sm + c * SC, SP, gA, gB, mlowA, recA, recB, tw);
        else         symbol_item<N, SYM, false>(sm + c * SC, SP, gA, gB, mlowA, recA, recB, tw);
    }
    __syncthreads();

    // ---- inverse pass 2
    if constexpr (P == 3) {
        constexpr int G2 = N / R2;
        for (int w = tid; w < NL * G2; w += T) {
            int c, g;
            if (VDIR) { c = w & (NL - 1); g = w >> lognl; } else { c = w / G2; g = w & (G2 - 1); }
            inv_pass_smem<N, R2, N / R1>(sm + c * SC, SP, g, tw);
        }
        __syncthreads();
    }

    // ---- inverse pass 1: shared -> registers -> global (+ delta-f source)
    for (int w = tid; w < NL * S1; w += T) {
        int c, t;
        if (VDIR) { c = w & (NL - 1); t = w >> lognl; } else { c = w / S1; t = w & (S1 - 1); }
        const float2* smc = sm + c * SC;
        float2 x[R1];
        x[0] = smc[padp(t) * SP];
#pragma unroll
        for (int q = 1; q < R1; ++q)
            x[brev(q, R1)] = cmulc(smc[padp(t + q * S1) * SP], __ldg(tw + t * q));
        idft_dit<R1, 1>(x);
        if (VDIR) {
            if (a.ng > 0) {
                const float sA = recs[(2 * c) * REC_WORDS + 19], sB = recs[(2 * c + 1) * REC_WORDS + 19];
#pragma unroll
                for (int g = 0; g < 4; ++g) {
                    if (g >= a.ng) break;
                    const float cg = a.cg[g];
                    const float* __restrict__ ft = a.feq_tab + (size_t)g * a.Nv;
                    const float* __restrict__ vt = a.vmu_tab + (size_t)g * a.Nv;
#pragma unroll
                    for (int k = 0; k < R1; ++k) {
                        const int j = t + k * S1;
                        const float fe = __ldg(ft + j), vm2 = 2.0f * __ldg(vt + j);
                        // f_eq,g(v - s) - f_eq,g(v) = f_eq,g(v) * expm1(c s (2(v-mu) - s))
                        x[k].x = fmaf(fe, expm1f(cg * sA * (vm2 - sA)), x[k].x);
                        x[k].y = fmaf(fe, expm1f(cg * sB * (vm2 - sB)), x[k].y);
                    }
                }
            }
#pragma unroll
            for (int k = 0; k < R1; ++k)
                __stcs(reinterpret_cast<float2*>(a.f + (size_t)(t + k * S1) * Nx + line0 + 2 * c), x[k]);
        } else {
            float* fa = a.f + (size_t)(line0 + 2 * c) * Nx + t;
#pragma unroll
            for (int k = 0; k < R1; ++k) { __stcs(fa + k * S1, x[k].x); __stcs(fa + Nx + k * S1, x[k].y); }
        }
    }
}

}  // namespace vog
