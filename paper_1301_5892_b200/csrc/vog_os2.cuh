// vog_os2.cuh -- overlap-save advection kernels, second generation (line length N >= 1024;
// SURVEY.md 8(a) S2-S7).  Product code; shares nothing with oracle/.
//
// Same method as vog_os.cuh (the circulant product of P:98-100 taken block-wise in Fourier space, P:131-149:
// blocks of LB = 256 samples of the rolled line, V = 224 kept, H = 16 discarded on either side), but the
// real-data trick is different.  The interpolation matrix is REAL, so two blocks A, B of the SAME line share
// the symbol lambda and can ride one complex transform:  z_n = A_n + i B_n,  Z = FFT_256(z),
// Z_k *= lambda_k (lambda_{256-k} = conj lambda_k),  z' = IFFT(Z)  =>  A' = Re z', B' = Im z'.
// Compared with the even/odd packing of vog_os.cuh there is no untangle / re-tangle stage, no "special"
// mirror item, no divergence, and a work item is ONE radix-16 butterfly (16 complex = 32 registers) in every
// phase, so the kernels fit 64 registers and run at twice the occupancy:
//   pass A   : item (pair, t):  n = t + 16 k  -> radix 16 over k, times W_256^{t k1}, stored at [k1][t]
//   middle   : item (pair, g = k1): radix 16 over t -> Z_{g + 16 k2}; times lambda; inverse radix 16
//   inverse A: item (pair, j): times conj W, inverse radix 16 over k1 -> z'_{j + 16 m}; m = 1..14 are the
//              kept samples of both blocks (uniform over the threads), stored straight to global memory.
// Every phase has 16 items per pair, every item touches only its own 16 scratch slots, and a thread lands
// (cp.async, 4 bytes: the full integer shift b of P:107 is applied by addressing, no alignment residue) exactly
// the samples that it transforms in pass A.
#pragma once
#include "vog_fft.cuh"
#include "vog_internal.h"

namespace vog {

namespace os2 {
constexpr int PW = 2 * OS_V;           // cells advanced by one pair of blocks (448)

__device__ __forceinline__ void cp_async4(void* smem, const void* gmem)
{
    const unsigned s = (unsigned)__cvta_generic_to_shared(smem);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4;\n" ::"r"(s), "l"(gmem) : "memory");
}
__device__ __forceinline__ void cp_async16(void* smem, const void* gmem)
{
    const unsigned s = (unsigned)__cvta_generic_to_shared(smem);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 16;\n" ::"r"(s), "l"(gmem) : "memory");
}
__device__ __forceinline__ void cp_async_wait_all()
{
    asm volatile("cp.async.commit_group;\ncp.async.wait_group 0;\n" ::: "memory");
}

// middle stage on 16 registers: x[j] = Y[g][j] -> Z_{g+16 q} at x[brev q] -> times lambda -> inverse over q.
// lam(k) returns lambda_k / 256 for k = 0..128 (the tabulated half); LS = stride of the table in float2.
template <int LS>
__device__ __forceinline__ void mid16(float2* x, const float2* __restrict__ lam, const int g)
{
    dft_dif<16, 1>(x);
#pragma unroll
    for (int q = 0; q < 8; ++q) x[brev(q, 16)] = cmul(x[brev(q, 16)], lam[(g + 16 * q) * LS]);
#pragma unroll
    for (int q = 8; q < 16; ++q) x[brev(q, 16)] = cmulc(x[brev(q, 16)], lam[(256 - 16 * q - g) * LS]);
    idft_dit<16, 1>(x);
}
}  // namespace os2

// ---------------------------------------------------------------------------------------------
// x-direction.  Scratch: 16 rows of 17 float2 per pair (2176 B): position p = 16 g + j sits at 17 g + j.
// All shared accesses are 8 bytes wide; passes A (16 lanes = 16 adjacent j of one row) and the middle stage
// (16 lanes = 16 rows, same j: bank pairs 2 g + 2 j mod 32) are bank-conflict free, and every address is
// "item base + compile-time constant" (no swizzle arithmetic, nothing to keep in registers).
// Persistent CTAs own whole lines (in place: all loads of a line group complete before the barrier that
// precedes its first store).
namespace os2 {
constexpr int XROW = 17;               // float2 per scratch row
constexpr int XPAIR = 16 * XROW;       // float2 per pair
}

__device__ __forceinline__ void osx2_land(float2* __restrict__ s, const float* __restrict__ gl, const int c0,
                                          const int mask)
{
    float* const sf = reinterpret_cast<float*>(s);
    if (c0 + OS_V + 241 <= mask + 1) {                 // the two windows do not wrap
        const float* p = gl + c0;
#pragma unroll
        for (int k = 0; k < 16; ++k) {
            os2::cp_async4(sf + 2 * os2::XROW * k, p + 16 * k);
            os2::cp_async4(sf + 2 * os2::XROW * k + 1, p + 16 * k + OS_V);
        }
    } else {
#pragma unroll 2
        for (int k = 0; k < 16; ++k) {
            os2::cp_async4(sf + 2 * os2::XROW * k, gl + ((c0 + 16 * k) & mask));
            os2::cp_async4(sf + 2 * os2::XROW * k + 1, gl + ((c0 + 16 * k + OS_V) & mask));
        }
    }
}

// s = pair base + t; tw = table + t
__device__ __forceinline__ void osx2_fwd(float2* __restrict__ s, const float2* __restrict__ tw)
{
    float2 x[16];
#pragma unroll
    for (int k = 0; k < 16; ++k) x[k] = s[os2::XROW * k];
    dft_dif<16, 1>(x);
    s[0] = x[0];
#pragma unroll
    for (int q = 1; q < 16; ++q) s[os2::XROW * q] = cmul(x[brev(q, 16)], tw[(q - 1) * 16]);
}

// s = pair base + 17 g
__device__ __forceinline__ void osx2_mid(float2* __restrict__ s, const int g, const float2* __restrict__ lam)
{
    float2 x[16];
#pragma unroll
    for (int j = 0; j < 16; ++j) x[j] = s[j];
    os2::mid16<1>(x, lam, g);
#pragma unroll
    for (int j = 0; j < 16; ++j) s[j] = x[j];
}

// inverse pass A of item (pair, j): kept samples m = 1..14 of block A (real parts) and block B (imaginary
// parts) go to cells o0 + 16 (m - 1) and o0 + OS_V + 16 (m - 1) of the line; cells >= N do not exist.
// s = pair base + j; tw = table + j
__device__ __forceinline__ void osx2_inv(float* __restrict__ gl, const int o0, const bool full, const int N,
                                         const float2* __restrict__ s, const float2* __restrict__ tw)
{
    float2 x[16];
    x[0] = s[0];
#pragma unroll
    for (int q = 1; q < 16; ++q) x[brev(q, 16)] = cmulc(s[os2::XROW * q], tw[(q - 1) * 16]);
    idft_dit<16, 1>(x);
    float* const o = gl + o0;
    if (full) {
#pragma unroll
        for (int m = 1; m < 15; ++m) {
            __stcs(o + 16 * (m - 1), x[m].x);
            __stcs(o + 16 * (m - 1) + OS_V, x[m].y);
        }
    } else {
#pragma unroll
        for (int m = 1; m < 15; ++m) {
            if (o0 + 16 * (m - 1) < N) __stcs(o + 16 * (m - 1), x[m].x);
            if (o0 + 16 * (m - 1) + OS_V < N) __stcs(o + 16 * (m - 1) + OS_V, x[m].y);
        }
    }
}

// One iteration = lpi whole lines = lpi * np pairs = 16 lpi np items per phase; blockDim.x is a multiple of 16,
// so the position index t = tid & 15 of a thread is the same for all its items.
template <int TMAX, int MINB>
__global__ void __launch_bounds__(TMAX, MINB) osx2_kernel(const OsArgs a)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int lpi = a.lpi, np = a.np, ptot = lpi * np, nitem = ptot * 16;
    float2* const scr = reinterpret_cast<float2*>(smem_raw);            // ptot * XPAIR
    float2* const lamS = scr + ptot * os2::XPAIR;                       // lpi rows of the symbol table
    float2* const twS = lamS + lpi * OS_LAMW;                           // 15 * 16
    const int tid = threadIdx.x, T = blockDim.x, t = tid & 15;
    const int N = a.N, mask = N - 1;
    const unsigned inv_np = a.inv_np;       // ceil(2^16 / np): pr / np == (pr * inv_np) >> 16 for pr < 2^12

    for (int i = tid; i < 240; i += T) twS[i] = __ldg(a.tw + i);

    // landing of item w of the line group that starts at line0, and of the group's table rows
    auto land = [&](const int w, const int line0) {
        const int pr = w >> 4;
        const int l = (int)(((unsigned)pr * inv_np) >> 16), pp = pr - l * np;
        const int line = line0 + l;
        if (line >= a.n_lines) return;
        const int b = __float_as_int(__ldg(&a.lam[(size_t)line * OS_LAMW + 129].x));
        osx2_land(scr + pr * os2::XPAIR + t, a.src + (size_t)line * N, (pp * os2::PW - OS_H + b + t) & mask, mask);
    };
    auto land_tab = [&](const int line0) {
        const int nl = min(lpi, a.n_lines - line0);
        const float4* src4 = reinterpret_cast<const float4*>(a.lam + (size_t)line0 * OS_LAMW);
        float4* dst4 = reinterpret_cast<float4*>(lamS);
        for (int i = tid; i < nl * (OS_LAMW / 2); i += T) os2::cp_async16(dst4 + i, src4 + i);
    };
    if ((int)blockIdx.x < a.n_groups) {
        for (int w = tid; w < nitem; w += T) land(w, blockIdx.x * lpi);
        land_tab(blockIdx.x * lpi);
    }
    __syncthreads();                               // twS visible
    for (int g = blockIdx.x; g < a.n_groups; g += gridDim.x) {
        const int line0 = g * lpi;
        os2::cp_async_wait_all();                  // this thread's samples (and table chunks) have landed
        // ---- pass A: every thread on the slots it landed itself
#pragma unroll 1
        for (int w = tid; w < nitem; w += T) {
            int tt = t;
            asm volatile("" : "+r"(tt));           // keep the 15 twiddle loads inside the loop (30 registers)
            osx2_fwd(scr + (w >> 4) * os2::XPAIR + t, twS + tt);
        }
        __syncthreads();
        // ---- middle stage
#pragma unroll 1
        for (int w = tid; w < nitem; w += T) {
            const int pr = w >> 4;
            const int l = (int)(((unsigned)pr * inv_np) >> 16);
            osx2_mid(scr + pr * os2::XPAIR + os2::XROW * t, t, lamS + l * OS_LAMW);
        }
        __syncthreads();
        // ---- inverse pass A: scratch -> registers -> global; the same item of the NEXT line group lands in
        // the slots just read.  In place this is safe: every load of THIS group completed before the
        // barrier after pass A, and the next group is other lines (owned by this CTA).
        const int gn = g + gridDim.x;
        if (gn < a.n_groups) land_tab(gn * lpi);   // lamS was last read before the barrier above
#pragma unroll 1
        for (int w = tid; w < nitem; w += T) {
            const int pr = w >> 4;
            const int l = (int)(((unsigned)pr * inv_np) >> 16), pp = pr - l * np;
            int tt = t;
            asm volatile("" : "+r"(tt));
            const float2* twp = twS + tt;
            if (line0 + l < a.n_lines)
                osx2_inv(a.dst + (size_t)(line0 + l) * N, pp * os2::PW + t, (pp + 1) * os2::PW <= N, N,
                         scr + pr * os2::XPAIR + t, twp);
            if (gn < a.n_groups) land(w, gn * lpi);
        }
    }
}

// ---------------------------------------------------------------------------------------------
// x-direction, register-landing variant (lines with at most 20 pairs, i.e. N <= 8192): one item per thread and
// phase (16 lpi np <= blockDim.x).  The 32 samples of a thread's pass-A item are loaded straight into the
// butterfly registers (coalesced 4-byte loads, 64-byte runs per half-warp) at the END of the previous
// iteration, so the scratch is only the exchange buffer between the phases (4 instead of 6 shared accesses
// per sample), and the 15 twiddles W^{t q} of a thread (t is fixed) are products of 4 register-resident
// powers W^t, W^2t, W^4t, W^8t instead of 15 shared loads per pass.
// ---------------------------------------------------------------------------------------------
// Block geometry of the default kernels (osx5_kernel, osv4_kernel) as template parameters: V kept samples per
// block, HLO discarded on the left, 256 - V - HLO on the right.  The cubic spline needs 16 + 16 (its circulant
// row decays like 0.268^|j|: section 6.1 of DESIGN.md), i.e. (224, 16); a Lagrange stencil of degree <= 17
// reaches 8 cells to the left and 9 to the right, so (232, 8) is exact for it and needs 5 % fewer
// blocks at 8192 (36 instead of 37) and 10 % fewer at 4096.
// Thread t of an inverse-pass item holds samples n = t + 16 m, m = 0..15; sample n is kept iff HLO <= n < HLO + V.
template <int V, int HLO, int M>
struct KeptM {
    static constexpr int lo = HLO - 16 * M, hi = HLO + V - 16 * M;     // kept iff lo <= t < hi
    static constexpr bool none = hi <= 0 || lo >= 16;
    static constexpr bool all = lo <= 0 && hi >= 16;
    static __device__ __forceinline__ bool kept(const int t) { return all || (!none && t >= lo && t < hi); }
};

// x: store the kept samples of both blocks of a pair.  o = line + (first cell of block A) + t - HLO, i.e. the cell
// of sample n = t; c = that cell index; cells >= N do not exist (checked only when !full).
template <int V, int HLO, int M = 0>
__device__ __forceinline__ void os2_store_x(float* __restrict__ o, const int c, const int N, const int t,
                                            const bool full, const float2* x)
{
    if constexpr (M < 16) {
        using K = KeptM<V, HLO, M>;
        if constexpr (!K::none) {
            const bool k = K::kept(t);
            if (k && (full || c + 16 * M < N)) __stcs(o + 16 * M, x[M].x);
            if (k && (full || c + 16 * M + V < N)) __stcs(o + 16 * M + V, x[M].y);
        }
        os2_store_x<V, HLO, M + 1>(o, c, N, t, full, x);
    }
}

// v: the same along rows (row stride Nx); po = column + (row of sample n = t) * Nx, r = that row.
template <int V, int HLO, int M = 0>
__device__ __forceinline__ void os2_store_v(float* __restrict__ po, const size_t Nx, const int r, const int Nv,
                                            const int t, const bool full, const float2* x)
{
    if constexpr (M < 16) {
        using K = KeptM<V, HLO, M>;
        if constexpr (!K::none) {
            const bool k = K::kept(t);
            if (k && (full || r + 16 * M < Nv)) __stcs(po + (size_t)(16 * M) * Nx, x[M].x);
            if (k && (full || r + 16 * M + V < Nv)) __stcs(po + (size_t)(16 * M + V) * Nx, x[M].y);
        }
        os2_store_v<V, HLO, M + 1>(po, Nx, r, Nv, t, full, x);
    }
}

struct Tw4 { float2 b1, b2, b4, b8; };

// Calls f(q, W^{t q}) for q = 1..15 (q a compile-time constant of each call), building the powers from the four
// binary ones (at most 3 chained roundings) in an order that keeps at most two temporaries alive.
template <int Q> struct QC { static constexpr int value = Q; };
template <class F>
__device__ __forceinline__ void os2_tw_each(const Tw4& w, F&& f)
{
    f(QC<1>(), w.b1); f(QC<2>(), w.b2); f(QC<4>(), w.b4); f(QC<8>(), w.b8);
    {
        const float2 y3 = cmul(w.b1, w.b2);
        f(QC<3>(), y3);
        f(QC<11>(), cmul(y3, w.b8));
        const float2 y7 = cmul(y3, w.b4);
        f(QC<7>(), y7);
        f(QC<15>(), cmul(y7, w.b8));
    }
    {
        const float2 y5 = cmul(w.b1, w.b4);
        f(QC<5>(), y5);
        f(QC<13>(), cmul(y5, w.b8));
    }
    {
        const float2 y6 = cmul(w.b2, w.b4);
        f(QC<6>(), y6);
        f(QC<14>(), cmul(y6, w.b8));
    }
    f(QC<9>(), cmul(w.b1, w.b8));
    f(QC<10>(), cmul(w.b2, w.b8));
    f(QC<12>(), cmul(w.b4, w.b8));
}

template <int V = OS_V>
__device__ __forceinline__ void osx3_load(float2* x, const float* __restrict__ gl, const int c0, const int mask)
{
    if (c0 + V + 241 <= mask + 1) {                    // the two windows do not wrap
        const float* p = gl + c0;
#pragma unroll
        for (int k = 0; k < 16; ++k) x[k] = make_float2(__ldg(p + 16 * k), __ldg(p + 16 * k + V));
    } else {
#pragma unroll
        for (int k = 0; k < 16; ++k)
            x[k] = make_float2(__ldg(gl + ((c0 + 16 * k) & mask)), __ldg(gl + ((c0 + 16 * k + V) & mask)));
    }
}

// RAW = false: the loads of a group are issued and consumed at the top of its own iteration (nothing is in
// flight while a CTA computes; the other CTAs of the SM cover for it).
// RAW = true: the lines of the NEXT group are copied as they are (cp.async, 16 bytes, no shift) into a raw line
// buffer right after pass A of the current group has emptied it, so they have the middle stage and the inverse
// pass to arrive (~2/3 of the time, 32 KB per CTA in flight); pass A then reads its samples from the raw
// buffer with the shift applied by addressing (4-byte shared loads, any alignment).  One more barrier per
// iteration (the raw lines are landed by all threads).
template <bool RAW>
__global__ void __launch_bounds__(320, 3) osx3_kernel(const OsArgs a)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int lpi = a.lpi, np = a.np, ptot = lpi * np, nitem = ptot * 16;
    float2* const scr = reinterpret_cast<float2*>(smem_raw);            // ptot * XPAIR
    float2* const lamS = scr + ptot * os2::XPAIR;                       // lpi rows of the symbol table
    float* const raw = reinterpret_cast<float*>(lamS + lpi * OS_LAMW);  // RAW: lpi lines of N floats
    const int tid = threadIdx.x, T = blockDim.x, t = tid & 15;
    const int N = a.N, mask = N - 1;
    const bool active = tid < nitem;
    const int pr = tid >> 4;
    const int l = (int)(((unsigned)pr * a.inv_np) >> 16), pp = pr - l * np;   // line of the group, pair of the line
    Tw4 w;
    w.b1 = __ldg(a.tw + t);               // [q-1][t] = e^{-2 pi i t q / 256}
    w.b2 = __ldg(a.tw + 16 + t);
    w.b4 = __ldg(a.tw + 3 * 16 + t);
    w.b8 = __ldg(a.tw + 7 * 16 + t);
    float2* const sA = scr + pr * os2::XPAIR + t;                       // passes A: column t of the pair
    float2* const sM = scr + pr * os2::XPAIR + os2::XROW * t;           // middle stage: row g = t
    const float2* const lamL = lamS + l * OS_LAMW;
    const int o0 = pp * os2::PW + t;
    const bool full = (pp + 1) * os2::PW <= N;
    const int G = gridDim.x;

    // the group's table rows and (RAW) its lines; a ragged last group has fewer lines
    auto land = [&](const int g) {
        const int line0 = g * lpi, nl = min(lpi, a.n_lines - line0);
        const float4* src4 = reinterpret_cast<const float4*>(a.lam + (size_t)line0 * OS_LAMW);
        float4* dst4 = reinterpret_cast<float4*>(lamS);
        for (int i = tid; i < nl * (OS_LAMW / 2); i += T) os2::cp_async16(dst4 + i, src4 + i);
        if constexpr (RAW) {
            const float4* s4 = reinterpret_cast<const float4*>(a.src + (size_t)line0 * N);
            float4* d4 = reinterpret_cast<float4*>(raw);
            const int n4 = nl * (N >> 2);
#pragma unroll 4
            for (int i = tid; i < n4; i += T) os2::cp_async16(d4 + i, s4 + i);
        }
    };
    if ((int)blockIdx.x < a.n_groups) land(blockIdx.x);
    for (int g = blockIdx.x; g < a.n_groups; g += G) {
        const int gn = g + G;
        const int line = min(g * lpi + l, a.n_lines - 1);      // (a ragged last group recomputes the last line)
        if constexpr (RAW) {
            os2::cp_async_wait_all();              // this thread's chunks of the raw lines and table rows
            __syncthreads();
        }
        // ---- pass A
        if (active) {
            float2 x[16];
            if constexpr (RAW) {
                const int b = __float_as_int(lamL[129].x);
                const float* const rl = raw + l * N;
                const int c0 = (pp * os2::PW - OS_H + b + t) & mask;
                if (c0 + OS_V + 241 <= N) {
#pragma unroll
                    for (int k = 0; k < 16; ++k) x[k] = make_float2(rl[c0 + 16 * k], rl[c0 + 16 * k + OS_V]);
                } else {
#pragma unroll
                    for (int k = 0; k < 16; ++k)
                        x[k] = make_float2(rl[(c0 + 16 * k) & mask], rl[(c0 + 16 * k + OS_V) & mask]);
                }
            } else {
                const int b = __float_as_int(__ldg(&a.lam[(size_t)line * OS_LAMW + 129].x));
                osx3_load(x, a.src + (size_t)line * N, (pp * os2::PW - OS_H + b + t) & mask, mask);
            }
            dft_dif<16, 1>(x);
            sA[0] = x[0];
            os2_tw_each(w, [&](auto qc, const float2 y) {
                constexpr int q = decltype(qc)::value;
                sA[os2::XROW * q] = cmul(x[brev(q, 16)], y);
            });
        }
        if constexpr (!RAW) os2::cp_async_wait_all();          // table rows
        __syncthreads();
        // ---- middle stage
        if (active) osx2_mid(sM, t, lamL);
        __syncthreads();
        // the raw buffer was emptied before the first barrier, the table rows were last read before the second:
        // the next group starts landing now and has the whole inverse pass (and the other CTAs' phases) to arrive
        if (gn < a.n_groups) land(gn);
        // ---- inverse pass A: scratch -> registers -> global.  In place this is safe: every load of THIS group
        // completed before the first barrier, and the other groups are other lines (owned by this CTA).
        if (active) {
            float2 x[16];
            x[0] = sA[0];
            os2_tw_each(w, [&](auto qc, const float2 y) {
                constexpr int q = decltype(qc)::value;
                x[brev(q, 16)] = cmulc(sA[os2::XROW * q], y);
            });
            idft_dit<16, 1>(x);
            if (g * lpi + l < a.n_lines) {
                float* const o = a.dst + (size_t)(g * lpi + l) * N + o0;
                if (full) {
#pragma unroll
                    for (int m = 1; m < 15; ++m) {
                        __stcs(o + 16 * (m - 1), x[m].x);
                        __stcs(o + 16 * (m - 1) + OS_V, x[m].y);
                    }
                } else {
#pragma unroll
                    for (int m = 1; m < 15; ++m) {
                        if (o0 + 16 * (m - 1) < N) __stcs(o + 16 * (m - 1), x[m].x);
                        if (o0 + 16 * (m - 1) + OS_V < N) __stcs(o + 16 * (m - 1) + OS_V, x[m].y);
                    }
                }
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------
// x-direction, warp-private variant.  The 16 items of a pair are 16 consecutive threads in EVERY phase (pass A
// item t, middle item g, inverse item j), so a warp owns its two pairs from the first load to the last store
// and the phases are separated by __syncwarp() only: the warps of a CTA drift apart freely and their load,
// compute and store phases overlap.  The symbol is read straight from the per-line table in global memory
// (a 1 KB row shared by all warps of the line: L1 hits), so nothing is staged CTA-wide.
// The only CTA-wide dependency left is the in-place hazard (every load of a line must complete before its
// first store): a split mbarrier -- each warp ARRIVES once its samples are in registers and WAITS just before
// its first store, with the middle stage and the inverse transform in between.  With INPLACE = false
// (src != dst) there is no synchronisation between warps at all.
namespace os2 {
__device__ __forceinline__ void mbar_init(unsigned long long* bar, const unsigned count)
{
    const unsigned s = (unsigned)__cvta_generic_to_shared(bar);
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" ::"r"(s), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(unsigned long long* bar)
{
    const unsigned s = (unsigned)__cvta_generic_to_shared(bar);
    asm volatile("{\n.reg .b64 st;\nmbarrier.arrive.shared::cta.b64 st, [%0];\n}\n" ::"r"(s) : "memory");
}
// (the suspend-time hint lets the hardware park the warp instead of spinning: in the first version 23 % of the
// kernel's instructions were this loop)
__device__ __forceinline__ void mbar_wait(unsigned long long* bar, const unsigned parity)
{
    const unsigned s = (unsigned)__cvta_generic_to_shared(bar);
    asm volatile(
        "{\n.reg .pred p;\nWAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1, %2;\n"
        "@!p bra WAIT_%=;\n}\n" ::"r"(s), "r"(parity), "r"(20000u) : "memory");
}
}  // namespace os2

template <bool INPLACE, int V, int HLO>
__global__ void __launch_bounds__(V == 232 ? 288 : 320, 3) osx5_kernel(const OsArgs a)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int lpi = a.lpi, np = a.np, ptot = lpi * np, nitem = ptot * 16;
    const int tid = threadIdx.x, T = blockDim.x, t = tid & 15, hw = tid >> 4;
    float2* const scr = reinterpret_cast<float2*>(smem_raw);            // ptot * XPAIR
    // one private copy of the line's table row per half-warp, or per warp when a group is one line (then both
    // pairs of a warp read the same copy: broadcast, and half the shared memory)
    const bool one_line = lpi == 1;
    float2* const lamP = scr + ptot * os2::XPAIR;
    unsigned long long* const bar = reinterpret_cast<unsigned long long*>(lamP + (one_line ? (T >> 5) : (T >> 4)) * OS_LAMW);
    const int N = a.N, mask = N - 1;
    Tw4 w;
    w.b1 = __ldg(a.tw + t);               // [q-1][t] = e^{-2 pi i t q / 256}
    w.b2 = __ldg(a.tw + 16 + t);
    w.b4 = __ldg(a.tw + 3 * 16 + t);
    w.b8 = __ldg(a.tw + 7 * 16 + t);
    float2* const lamL = lamP + (one_line ? (hw >> 1) : hw) * OS_LAMW;
    const int cp0 = one_line ? (tid & 31) : t, cps = one_line ? 32 : 16;      // this thread's chunks of the copy
    if constexpr (INPLACE) {
        if (tid == 0) os2::mbar_init(bar, T >> 5);
        __syncthreads();
    }
    pdl_wait();                                   // (the twiddles above are plan constants; tables and grid are not)
    pdl_launch_dependents();
    unsigned parity = 0;
    // A line group has nitem items; thread tid takes items tid, tid + T, .. ("rounds"; one round when the group
    // fits the CTA, two for 16384-cell lines).  Per round: load, pass A, middle stage -- the pair's spectrum
    // stays in its scratch; then, once every load of the group has completed, per round: inverse pass and stores.
    for (int g = blockIdx.x; g < a.n_groups; g += gridDim.x) {
#pragma unroll 1
        for (int it = tid; it - (tid & 31) < nitem; it += T) {          // (trip count uniform over the warp)
            const int pr = it >> 4;
            const bool active = it < nitem;
            const int l = (int)(((unsigned)pr * a.inv_np) >> 16), pp = pr - l * np;   // line of the group, pair of the line
            const int line = min(g * lpi + l, a.n_lines - 1);  // (a ragged last group recomputes the last line)
            const float2* __restrict__ lamG = a.lam + (size_t)line * OS_LAMW;
            float2* const sA = scr + pr * os2::XPAIR + t;                       // passes A: column t of the pair
            float2* const sM = scr + pr * os2::XPAIR + os2::XROW * t;           // middle stage: row g = t
            // ---- pass A straight from global memory
            // the (half-)warp's copy of the line's symbol table lands behind pass A (its previous contents were
            // last read by these threads before the __syncwarp() that closed their last middle stage); with one
            // line per group all 32 lanes copy, the inactive ones of the last warp included
            if (active || one_line) {
                const float2* __restrict__ lamC = one_line ? a.lam + (size_t)min(g, a.n_lines - 1) * OS_LAMW : lamG;
                for (int i = cp0; i < OS_LAMW / 2; i += cps)
                    os2::cp_async16(reinterpret_cast<float4*>(lamL) + i, reinterpret_cast<const float4*>(lamC) + i);
            }
            if (active) {
                float2 x[16];
                const int b = __float_as_int(__ldg(&lamG[129].x));
                osx3_load<V>(x, a.src + (size_t)line * N, (pp * (2 * V) - HLO + b + t) & mask, mask);
                dft_dif<16, 1>(x);
                sA[0] = x[0];
                os2_tw_each(w, [&](auto qc, const float2 y) {
                    constexpr int q = decltype(qc)::value;
                    sA[os2::XROW * q] = cmul(x[brev(q, 16)], y);
                });
            }
            os2::cp_async_wait_all();
            __syncwarp();
            // (the shared stores of pass A needed every loaded value, and a warp issues in order: once its last
            // round is here, all loads of this warp have completed)
            if constexpr (INPLACE) {
                if (it - (tid & 31) + T >= nitem && (tid & 31) == 0) os2::mbar_arrive(bar);
            }
            // ---- middle stage
            if (active) {
                float2 x[16];
#pragma unroll
                for (int j = 0; j < 16; ++j) x[j] = sM[j];
                os2::mid16<1>(x, lamL, t);
#pragma unroll
                for (int j = 0; j < 16; ++j) sM[j] = x[j];
            }
            __syncwarp();
        }
        if constexpr (INPLACE) {                   // every load of the group has completed, in every warp
            os2::mbar_wait(bar, parity);
            parity ^= 1u;
        }
        // ---- inverse pass A: scratch -> registers -> global
#pragma unroll 1
        for (int it = tid; it < nitem; it += T) {
            const int pr = it >> 4;
            const int l = (int)(((unsigned)pr * a.inv_np) >> 16), pp = pr - l * np;
            const float2* const sA = scr + pr * os2::XPAIR + t;
            float2 x[16];
            x[0] = sA[0];
            os2_tw_each(w, [&](auto qc, const float2 y) {
                constexpr int q = decltype(qc)::value;
                x[brev(q, 16)] = cmulc(sA[os2::XROW * q], y);
            });
            idft_dit<16, 1>(x);
            if (g * lpi + l < a.n_lines) {
                const int c = pp * (2 * V) + t - HLO;          // cell of sample n = t of block A
                os2_store_x<V, HLO>(a.dst + (size_t)(g * lpi + l) * N + c, c, N, t, (pp + 1) * (2 * V) <= N, x);
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------
// v-direction.  A strip is 32 adjacent columns = the 32 lanes of a warp; every lane advects ITS column, the
// pair = two consecutive row blocks of that column.  A row of the strip is one 128-byte line: loads and
// stores are fully coalesced, and a lane applies its own integer shift b_c by addressing.  Scratch is
// [position][lane] float2 (64 KB per pair): conflict-free with no padding; an item (t, g or j) is one WARP, so
// a CTA of 16 warps does each phase of a pair in one round.  The symbol tables arrive transposed
// ([k][column]) and are staged once per CTA; CTAs loop over gpc pairs.  Out of place (src != dst).
// Landing is planar inside the 256 bytes of a position (32 real parts = block A, then 32 imaginary parts =
// block B) so that the 4-byte copies of a warp are bank-conflict free; pass A reads the planar words and
// writes the position back as interleaved float2 (all reads of the warp precede its writes).
__device__ __forceinline__ void osv2_land(float* __restrict__ pw, const float* __restrict__ col, const int Nx,
                                          const int vmask, const int r0)
{
    constexpr int PS = 16 * 32 * 2;                 // floats between positions t + 16 k and t + 16 (k + 1)
    const int rr = r0 & vmask;
    if (rr + OS_V + 241 <= vmask + 1) {             // the two windows do not wrap: constant row stride
        const float* p = col + (size_t)rr * Nx;
        const float* q = p + (size_t)OS_V * Nx;
        const size_t s16 = (size_t)16 * Nx;
#pragma unroll
        for (int k = 0; k < 16; ++k) {
            os2::cp_async4(pw + k * PS, p);
            os2::cp_async4(pw + k * PS + 32, q);
            p += s16;
            q += s16;
        }
    } else {
#pragma unroll
        for (int k = 0; k < 16; ++k) {
            const int ra = (r0 + 16 * k) & vmask, rb = (r0 + 16 * k + OS_V) & vmask;
            os2::cp_async4(pw + k * PS, col + (size_t)ra * Nx);
            os2::cp_async4(pw + k * PS + 32, col + (size_t)rb * Nx);
        }
    }
}

// delta-f source on the samples of one item: x[m].x += f_eq,g(v_j)(e^{X_j} - 1) at rows j = r0 + 16 m
// (r0 = row of sample n = t of block A), x[m].y the same at rows j + V, with X_j = c s (2 (v_j - mu) - s) affine in j.
// Along rows 16 apart expm1 obeys e' = e R + r (R = e^h, r = expm1(h), h = 32 c s dv); the recurrence starts in
// the middle (m = 8) and runs both ways (RS[g] = (R, r, 1/R, expm1(-h)) per lane), so at most 8 steps accumulate.
// Samples that are not kept (m = 15, and m = 0 unless HLO < 16) are skipped or harmlessly updated.  The f_eq table
// has 512 floats of padding: rows >= Nv are read but never stored; rows < 0 (m = 0 of the first pair) are clamped.
template <int V, int HLO>
__device__ __forceinline__ void osv2_source(float2* x, const OsArgs& a, const float4* __restrict__ RS, const int lane,
                                            const int r0, const float ssh)
{
    constexpr int M0 = HLO < 16 ? 0 : 1;
#pragma unroll 1
    for (int g = 0; g < a.ng; ++g) {
        const float cgs = a.cg4[g] * ssh;
        const float* __restrict__ fa = a.feq_tab + g * a.Nv + r0;
        const float u0 = __ldg(a.vmu_tab + g * a.Nv);                          // v_0 - mu_g
        const float4 Rr = RS[g * 32 + lane];
        const float ea8 = expm1f(cgs * (2.0f * fmaf((float)(r0 + 128), a.dvf, u0) - ssh));
        const float eb8 = expm1f(cgs * (2.0f * fmaf((float)(r0 + 128 + V), a.dvf, u0) - ssh));
        float ea = ea8, eb = eb8;
#pragma unroll
        for (int m = 8; m < 15; ++m) {
            x[m].x = fmaf(__ldg(fa + 16 * m), ea, x[m].x);
            x[m].y = fmaf(__ldg(fa + 16 * m + V), eb, x[m].y);
            ea = fmaf(ea, Rr.x, Rr.y);
            eb = fmaf(eb, Rr.x, Rr.y);
        }
        ea = ea8; eb = eb8;
#pragma unroll
        for (int m = 7; m >= M0; --m) {
            ea = fmaf(ea, Rr.z, Rr.w);
            eb = fmaf(eb, Rr.z, Rr.w);
            const int ia = (m == 0) ? max(-r0, 0) : 16 * m;      // (row r0 < 0 exists only as a discarded sample)
            x[m].x = fmaf(__ldg(fa + ia), ea, x[m].x);
            x[m].y = fmaf(__ldg(fa + 16 * m + V), eb, x[m].y);
        }
    }
}

__global__ void __launch_bounds__(512, 2) osv2_kernel(const OsArgs a)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    constexpr int W = 32;
    float2* const scr = reinterpret_cast<float2*>(smem_raw);                  // 256 * 32
    float2* const lamS = scr + 256 * W;                                       // 130 * 32, [k][lane]
    float2* const twS = lamS + OS_LAMW * W;                                   // 15 * 16
    float4* const RS = reinterpret_cast<float4*>(twS + 240);                  // [4][32] source recurrence constants
    const int tid = threadIdx.x, T = blockDim.x, lane = tid & 31, wid = tid >> 5;   // wid = item index (t, g, j)
    const int Nx = a.Nx, Nv = a.Nv, vmask = Nv - 1;
    const int c0 = blockIdx.x * W;

    {   // symbol tables of the 32 columns: 130 rows of 256 B, transposed layout [k][column]
        const float4* src4 = reinterpret_cast<const float4*>(a.lam + c0);
        float4* dst4 = reinterpret_cast<float4*>(lamS);
        for (int i = tid; i < OS_LAMW * 16; i += T)
            os2::cp_async16(dst4 + i, src4 + (size_t)(i >> 4) * (Nx / 2) + (i & 15));
    }
    for (int i = tid; i < 240; i += T) twS[i] = __ldg(a.tw + i);
    os2::cp_async_wait_all();
    __syncthreads();
    const int b = __float_as_int(lamS[129 * W + lane].x);
    const float ssh = lamS[129 * W + lane].y;
    if (a.ng > 0 && tid < 4 * W) {
        // delta-f source: x_j = c s (2 (v_j - mu) - s) is affine in the row j, so along rows 16 apart
        // expm1 obeys e' = e R + r with R = exp(h), r = expm1(h), h = 32 c s dv
        const int g = tid >> 5;
        const float h = 32.0f * (g < a.ng ? a.cg4[g] : 0.0f) * ssh * a.dvf;
        RS[g * W + lane] = make_float4(expf(h), expm1f(h), expf(-h), expm1f(-h));
    }
    const float* const col = a.src + c0 + lane;
    float* const ocol = a.dst + c0 + lane;
    const int p0 = blockIdx.y * a.gpc, p1 = min(a.np, p0 + a.gpc);
    float* const pw = reinterpret_cast<float*>(scr + wid * W) + lane;        // planar words of position t = wid
    float2* const own = scr + wid * W + lane;                                 // the same position, interleaved
    constexpr int PS2 = 16 * W;                                               // float2 between positions 16 apart

    if (p0 < p1) osv2_land(pw, col, Nx, vmask, p0 * os2::PW - OS_H + b + wid);
    __syncthreads();                               // RS visible (twS, lamS already are)
    for (int p = p0; p < p1; ++p) {
        int wt = wid;
        asm volatile("" : "+r"(wt));               // keep the twiddle loads inside the loop (30 registers)
        const float2* const twp = twS + wt;
        os2::cp_async_wait_all();                  // this thread's samples have landed
        // ---- pass A (item t = wid)
        {
            float2 x[16];
#pragma unroll
            for (int k = 0; k < 16; ++k) x[k] = make_float2(pw[k * PS2 * 2], pw[k * PS2 * 2 + W]);
            __syncwarp();                          // planar words all read before the interleaved writes
            dft_dif<16, 1>(x);
            own[0] = x[0];
#pragma unroll
            for (int q = 1; q < 16; ++q) own[q * PS2] = cmul(x[brev(q, 16)], twp[(q - 1) * 16]);
        }
        __syncthreads();
        // ---- middle stage (item g = wid): positions 16 g + j
        {
            float2* const s = scr + wid * 16 * W + lane;
            float2 x[16];
#pragma unroll
            for (int j = 0; j < 16; ++j) x[j] = s[j * W];
            os2::mid16<W>(x, lamS + lane, wid);
#pragma unroll
            for (int j = 0; j < 16; ++j) s[j * W] = x[j];
        }
        __syncthreads();
        // ---- inverse pass A (item j = wid): kept samples m = 1..14 -> rows p PW + j + 16 (m - 1) (+ OS_V)
        {
            float2 x[16];
            x[0] = own[0];
#pragma unroll
            for (int q = 1; q < 16; ++q) x[brev(q, 16)] = cmulc(own[q * PS2], twp[(q - 1) * 16]);
            __syncwarp();                          // interleaved words all read before the next planar landing
            if (p + 1 < p1) osv2_land(pw, col, Nx, vmask, (p + 1) * os2::PW - OS_H + b + wid);
            idft_dit<16, 1>(x);
            const int row0 = p * os2::PW + wid;    // row of m = 1, block A
            if (a.ng > 0) osv2_source<OS_V, OS_H>(x, a, RS, lane, row0 - 16, ssh);
            float* po = ocol + (size_t)row0 * Nx;
            const size_t s16 = (size_t)16 * Nx, sV = (size_t)OS_V * Nx;
            if (p * os2::PW + os2::PW <= Nv) {
#pragma unroll
                for (int m = 1; m < 15; ++m) {
                    __stcs(po, x[m].x);
                    __stcs(po + sV, x[m].y);
                    po += s16;
                }
            } else {
#pragma unroll
                for (int m = 1; m < 15; ++m) {
                    if (row0 + 16 * (m - 1) < Nv) __stcs(po, x[m].x);
                    if (row0 + 16 * (m - 1) + OS_V < Nv) __stcs(po + sV, x[m].y);
                    po += s16;
                }
            }
        }
        // no barrier here: pass A touches only the warp's own positions
    }
}

// ---------------------------------------------------------------------------------------------
// v-direction, register-landing variant: as osv2_kernel, but the 32 samples of a warp's pass-A item go
// straight from global memory into the butterfly registers (each load instruction of a warp is one
// 128-byte row segment per distinct shift), and the twiddles are products of four register-resident powers
// (t = warp index is fixed).  The scratch is only the exchange buffer between the phases.
__device__ __forceinline__ void osv3_load(float2* x, const float* __restrict__ col, const int Nx, const int vmask,
                                          const int r0)
{
    const int rr = r0 & vmask;
    if (rr + OS_V + 241 <= vmask + 1) {             // the two windows do not wrap: constant row stride
        const float* p = col + (size_t)rr * Nx;
        const float* q = p + (size_t)OS_V * Nx;
        const size_t s16 = (size_t)16 * Nx;
#pragma unroll
        for (int k = 0; k < 16; ++k) {
            x[k] = make_float2(__ldg(p), __ldg(q));
            p += s16;
            q += s16;
        }
    } else {
#pragma unroll
        for (int k = 0; k < 16; ++k) {
            const int ra = (r0 + 16 * k) & vmask, rb = (r0 + 16 * k + OS_V) & vmask;
            x[k] = make_float2(__ldg(col + (size_t)ra * Nx), __ldg(col + (size_t)rb * Nx));
        }
    }
}

__global__ void __launch_bounds__(512, 2) osv3_kernel(const OsArgs a)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    constexpr int W = 32;
    float2* const scr = reinterpret_cast<float2*>(smem_raw);                  // 256 * 32
    float2* const lamS = scr + 256 * W;                                       // 130 * 32, [k][lane]
    float4* const RS = reinterpret_cast<float4*>(lamS + OS_LAMW * W);         // [4][32] source recurrence constants
    const int tid = threadIdx.x, T = blockDim.x, lane = tid & 31, wid = tid >> 5;   // wid = item index (t, g, j)
    const int Nx = a.Nx, Nv = a.Nv, vmask = Nv - 1;
    const int c0 = blockIdx.x * W;

    {   // symbol tables of the 32 columns: 130 rows of 256 B, transposed layout [k][column]
        const float4* src4 = reinterpret_cast<const float4*>(a.lam + c0);
        float4* dst4 = reinterpret_cast<float4*>(lamS);
        for (int i = tid; i < OS_LAMW * 16; i += T)
            os2::cp_async16(dst4 + i, src4 + (size_t)(i >> 4) * (Nx / 2) + (i & 15));
    }
    Tw4 w;
    w.b1 = __ldg(a.tw + wid);
    w.b2 = __ldg(a.tw + 16 + wid);
    w.b4 = __ldg(a.tw + 3 * 16 + wid);
    w.b8 = __ldg(a.tw + 7 * 16 + wid);
    // integer shift and source shift of this lane's column straight from the table in global memory, so that
    // the first loads do not wait for the staged copy
    const float2 e129 = __ldg(a.lam + (size_t)129 * Nx + c0 + lane);
    const int b = __float_as_int(e129.x);
    const float ssh = e129.y;
    if (a.ng > 0 && tid < 4 * W) {
        const int g = tid >> 5;
        const float h = 32.0f * (g < a.ng ? a.cg4[g] : 0.0f) * ssh * a.dvf;
        RS[g * W + lane] = make_float4(expf(h), expm1f(h), expf(-h), expm1f(-h));
    }
    const float* const col = a.src + c0 + lane;
    float* const ocol = a.dst + c0 + lane;
    const int p0 = blockIdx.y * a.gpc, p1 = min(a.np, p0 + a.gpc);
    float2* const own = scr + wid * W + lane;                                 // position t = wid
    constexpr int PS2 = 16 * W;                                               // float2 between positions 16 apart

    for (int p = p0; p < p1; ++p) {
        // ---- pass A (item t = wid) straight from global memory
        {
            float2 x[16];
            osv3_load(x, col, Nx, vmask, p * os2::PW - OS_H + b + wid);
            dft_dif<16, 1>(x);
            own[0] = x[0];
            os2_tw_each(w, [&](auto qc, const float2 y) {
                constexpr int q = decltype(qc)::value;
                own[q * PS2] = cmul(x[brev(q, 16)], y);
            });
        }
        if (p == p0) os2::cp_async_wait_all();     // symbol tables
        __syncthreads();
        // ---- middle stage (item g = wid): positions 16 g + j
        {
            float2* const s = scr + wid * 16 * W + lane;
            float2 x[16];
#pragma unroll
            for (int j = 0; j < 16; ++j) x[j] = s[j * W];
            os2::mid16<W>(x, lamS + lane, wid);
#pragma unroll
            for (int j = 0; j < 16; ++j) s[j * W] = x[j];
        }
        __syncthreads();
        // ---- inverse pass A (item j = wid): kept samples m = 1..14 -> rows p PW + j + 16 (m - 1) (+ OS_V)
        {
            float2 x[16];
            x[0] = own[0];
            os2_tw_each(w, [&](auto qc, const float2 y) {
                constexpr int q = decltype(qc)::value;
                x[brev(q, 16)] = cmulc(own[q * PS2], y);
            });
            idft_dit<16, 1>(x);
            const int row0 = p * os2::PW + wid;    // row of m = 1, block A
            if (a.ng > 0) osv2_source<OS_V, OS_H>(x, a, RS, lane, row0 - 16, ssh);
            float* po = ocol + (size_t)row0 * Nx;
            const size_t s16 = (size_t)16 * Nx, sV = (size_t)OS_V * Nx;
            if (p * os2::PW + os2::PW <= Nv) {
#pragma unroll
                for (int m = 1; m < 15; ++m) {
                    __stcs(po, x[m].x);
                    __stcs(po + sV, x[m].y);
                    po += s16;
                }
            } else {
#pragma unroll
                for (int m = 1; m < 15; ++m) {
                    if (row0 + 16 * (m - 1) < Nv) __stcs(po, x[m].x);
                    if (row0 + 16 * (m - 1) + OS_V < Nv) __stcs(po + sV, x[m].y);
                    po += s16;
                }
            }
        }
        // no barrier here: the next pass A writes only the warp's own positions, which it has just read
    }
}

// ---------------------------------------------------------------------------------------------
// v-direction, coalesced-landing variant.  osv2_kernel lets every lane fetch its own shifted rows, which is a
// gather of up to 32 rows per load instruction when neighbouring columns have different integer shifts (the
// sweep's random shifts).  Here the CTA first copies the UNION of the rows its 32 columns need -- unshifted,
// 16 bytes per lane, whole 128-byte row segments -- into shared memory, raw[row][column], and a lane applies its
// own shift when it reads its samples from there: in this layout a lane only ever touches its own bank, so
// any per-lane row offset is conflict-free.  The raw rows (480 + R, R = spread of the shifts in the strip,
// <= 32) share the 64 KB of the exchange buffer, so two more barriers separate "raw read" from "exchange
// written".  Strips whose shifts spread over more than 32 rows fall back to the per-lane fetch (same layout).
template <int V, int HLO>
__global__ void __launch_bounds__(512, 2) osv4_kernel(const OsArgs a)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    constexpr int W = 32;
    float2* const scr = reinterpret_cast<float2*>(smem_raw);                  // 256 * 32 float2 = raw[512][32] floats
    float* const raw = reinterpret_cast<float*>(smem_raw);
    float2* const lamS = scr + 256 * W;                                       // 130 * 32, [k][lane]
    float2* const twS = lamS + OS_LAMW * W;                                   // 15 * 16
    float4* const RS = reinterpret_cast<float4*>(twS + 240);                  // [4][32] source recurrence constants
    const int tid = threadIdx.x, T = blockDim.x, lane = tid & 31, wid = tid >> 5;   // wid = item index (t, g, j)
    const int Nx = a.Nx, Nv = a.Nv, vmask = Nv - 1;
    const int c0 = blockIdx.x * W;

    for (int i = tid; i < 240; i += T) twS[i] = __ldg(a.tw + i);             // (plan constant: before the wait)
    pdl_wait();                                   // the symbol tables and the source grid come from earlier kernels
    pdl_launch_dependents();
    {   // symbol tables of the 32 columns: 130 rows of 256 B, transposed layout [k][column]
        const float4* src4 = reinterpret_cast<const float4*>(a.lam + c0);
        float4* dst4 = reinterpret_cast<float4*>(lamS);
        for (int i = tid; i < OS_LAMW * 16; i += T)
            os2::cp_async16(dst4 + i, src4 + (size_t)(i >> 4) * (Nx / 2) + (i & 15));
    }
    // integer shift (rows) and source shift of this lane's column
    const float2 e129 = __ldg(a.lam + (size_t)129 * Nx + c0 + lane);
    const int b = __float_as_int(e129.x);
    const float ssh = e129.y;
    // spread of the shifts over the strip, as signed distances from column 0's (shifts live mod Nv)
    const int b0 = __shfl_sync(0xffffffffu, b, 0);
    int d = (((b - b0) + (Nv >> 1)) & vmask) - (Nv >> 1);
    int dmin = d, dmax = d;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        dmin = min(dmin, __shfl_xor_sync(0xffffffffu, dmin, o));
        dmax = max(dmax, __shfl_xor_sync(0xffffffffu, dmax, o));
    }
    const int R = dmax - dmin;
    constexpr int RMAX = 512 - OS_LB - V;          // the raw rows (V + 256 + R) share the 512 rows of the exchange buffer
    const bool gather = R > RMAX;             // uniform over the CTA (every warp sees the same 32 columns)
    const int db = gather ? 0 : d - dmin;          // this lane's row offset inside the raw window
    const int base = gather ? b : b0 + dmin;       // first raw row = pair start - HLO + base
    if (a.ng > 0 && tid < 4 * W) {
        const int g = tid >> 5;
        const float h = 32.0f * (g < a.ng ? a.cg4[g] : 0.0f) * ssh * a.dvf;
        RS[g * W + lane] = make_float4(expf(h), expm1f(h), expf(-h), expm1f(-h));
    }
    const float* const col = a.src + c0 + lane;
    float* const ocol = a.dst + c0 + lane;
    const int p0 = blockIdx.y * a.gpc, p1 = min(a.np, p0 + a.gpc);
    float2* const own = scr + wid * W + lane;                                 // position t = wid, interleaved
    constexpr int PS2 = 16 * W;                                               // float2 between positions 16 apart
    const int nrows = V + OS_LB + (gather ? 0 : R);

    for (int p = p0; p < p1; ++p) {
        // ---- landing: the union of the rows, unshifted (or, in the fallback, every lane its own rows)
        const int rs = p * (2 * V) - HLO + base;
        if (!gather) {
            const float* const src = a.src + c0;
            for (int c = tid; c < nrows * 8; c += T) {
                const int r = c >> 3, q4 = (c & 7) * 4;
                os2::cp_async16(raw + r * W + q4, src + (size_t)((rs + r) & vmask) * Nx + q4);
            }
        } else {
            for (int r = wid; r < nrows; r += 16) os2::cp_async4(raw + r * W + lane, col + (size_t)((rs + r) & vmask) * Nx);
        }
        os2::cp_async_wait_all();
        __syncthreads();
        // ---- pass A (item t = wid): samples from the raw rows with this lane's offset
        {
            float2 x[16];
            const float* const rp = raw + (wid + db) * W + lane;
#pragma unroll
            for (int k = 0; k < 16; ++k) x[k] = make_float2(rp[16 * k * W], rp[(16 * k + V) * W]);
            __syncthreads();                       // raw rows all read before the exchange buffer is written
            const float2* const twp = twS + wid;
            dft_dif<16, 1>(x);
            own[0] = x[0];
#pragma unroll
            for (int q = 1; q < 16; ++q) own[q * PS2] = cmul(x[brev(q, 16)], twp[(q - 1) * 16]);
        }
        __syncthreads();
        // ---- middle stage (item g = wid): positions 16 g + j
        {
            float2* const s = scr + wid * 16 * W + lane;
            float2 x[16];
#pragma unroll
            for (int j = 0; j < 16; ++j) x[j] = s[j * W];
            os2::mid16<W>(x, lamS + lane, wid);
#pragma unroll
            for (int j = 0; j < 16; ++j) s[j * W] = x[j];
        }
        __syncthreads();
        // ---- inverse pass A (item j = wid): kept samples m = 1..14 -> rows p PW + j + 16 (m - 1) (+ OS_V)
        {
            float2 x[16];
            const float2* const twp = twS + wid;
            x[0] = own[0];
#pragma unroll
            for (int q = 1; q < 16; ++q) x[brev(q, 16)] = cmulc(own[q * PS2], twp[(q - 1) * 16]);
            idft_dit<16, 1>(x);
            const int r0 = p * (2 * V) + wid - HLO;        // row of sample n = t = wid of block A
            if (a.ng > 0) osv2_source<V, HLO>(x, a, RS, lane, r0, ssh);
            os2_store_v<V, HLO>(ocol + (ptrdiff_t)r0 * Nx, (size_t)Nx, r0, Nv, wid, (p + 1) * (2 * V) <= Nv, x);
        }
        if (p + 1 < p1) __syncthreads();           // the exchange buffer is read before the next raw rows land
    }
}

}  // namespace vog
